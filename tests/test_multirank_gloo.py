"""World-size-2 run of the data-parallel path on CPU (gloo): each rank takes its batch shard, runs the
operator on it (here: the oracle stands in for the per-rank kernel call), and the shared weight gradients are
summed with ONE all-reduce -- the result must equal the unsharded run."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_27229_b200 import shard, synth


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ.setdefault("OMP_NUM_THREADS", "2")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import carve_oracle as orc
    cfg = synth.Config("t", B=3, H=2, T=64, L=16, dk=64, dv=64, r=8, dtype="f32", wstd=0.2, s0_std=0.1, seed=3)
    x, ct = synth.make_inputs(cfg, with_decay_params=True), synth.make_cotangents(cfg)
    xs, cts = shard.shard_batch(x, rank, world), shard.shard_batch(ct, rank, world)
    lo, hi = shard.batch_range(cfg.B, rank, world)
    s = orc.Shape(B=hi - lo, H=cfg.H, T=cfg.T, L=cfg.L, dk=cfg.dk, dv=cfg.dv, r=cfg.r)
    O, Sf = orc.fwd(s, xs)
    g = orc.bwd(s, xs, cts["dO"], cts["dS_final"])
    buf = torch.from_numpy(shard.pack_weight_grads(g))
    dist.all_reduce(buf)                                    # the only collective of the path
    g.update(shard.unpack_weight_grads(buf.numpy(), g))
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), O=O, Sf=Sf, **g)
    dist.destroy_process_group()


def test_two_rank_sharding_matches_unsharded(oracle, tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    cfg = synth.Config("t", B=3, H=2, T=64, L=16, dk=64, dv=64, r=8, dtype="f32", wstd=0.2, s0_std=0.1, seed=3)
    x, ct = synth.make_inputs(cfg, with_decay_params=True), synth.make_cotangents(cfg)
    s = oracle.Shape(B=cfg.B, H=cfg.H, T=cfg.T, L=cfg.L, dk=cfg.dk, dv=cfg.dv, r=cfg.r)
    O, Sf = oracle.fwd(s, x)
    g = oracle.bwd(s, x, ct["dO"], ct["dS_final"])
    parts = [np.load(os.path.join(tmp_path, f"rank{r}.npz")) for r in range(world)]
    assert np.array_equal(np.concatenate([p["O"] for p in parts]), O)
    assert np.array_equal(np.concatenate([p["Sf"] for p in parts]), Sf)
    for n in ("dq", "dk", "dv", "df", "dbx", "dwx", "dbeta", "dS0"):
        assert np.array_equal(np.concatenate([p[n] for p in parts]), g[n]), n
    for n in shard.WEIGHT_GRADS:                            # summed in a different order: equal to rounding
        for p in parts:
            assert np.allclose(p[n], g[n], rtol=1e-12, atol=1e-14), n


def test_batch_range_partitions():
    for B in (1, 3, 8, 13):
        for world in (1, 2, 4, 8):
            r = [shard.batch_range(B, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == B
            assert all(r[i][1] == r[i + 1][0] for i in range(world - 1))
