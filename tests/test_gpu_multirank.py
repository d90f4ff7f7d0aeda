"""Two ranks on two GPUs with the REAL kernels: each rank runs carve_fwd + carve_bwd on its batch shard, the packed weight
gradients are summed with one NCCL all-reduce, and the result is compared with the unsharded call on rank 0.
Skipped when fewer than two CUDA devices are visible (every box of this run has one); the sharding logic itself is
covered on CPU by tests/test_multirank_gloo.py."""
import os
import socket

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist
    from paper_2606_27229_b200 import carve, shard, synth
    from tests.gpu_util import params_of, run_bwd, run_fwd
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    cfg = synth.Config("t", B=4, H=2, T=256, L=64, dk=128, dv=128, r=16, dtype="bf16", wstd=0.1, seed=5)
    x, ct = synth.make_inputs(cfg), synth.make_cotangents(cfg)
    xs, cts = shard.shard_batch(x, rank, world), shard.shard_batch(ct, rank, world)
    lo, hi = shard.batch_range(cfg.B, rank, world)
    p = params_of(cfg.with_(B=hi - lo))
    O, Sf, h = run_fwd(p, xs, need_bwd=True)
    g, gd = run_bwd(p, h, cts)
    buf = torch.cat([gd[n].reshape(-1) for n in shard.WEIGHT_GRADS])
    dist.all_reduce(buf)                                     # the only collective of the path
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), O=O, wg=buf.cpu().numpy().astype(np.float64), dq=g["dq"])
    dist.destroy_process_group()


def test_two_gpu_sharded_matches_unsharded(tmp_path):
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    import torch.multiprocessing as mp
    from paper_2606_27229_b200 import shard, synth
    from tests.gpu_util import params_of, run_bwd, run_fwd
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    cfg = synth.Config("t", B=4, H=2, T=256, L=64, dk=128, dv=128, r=16, dtype="bf16", wstd=0.1, seed=5)
    x, ct = synth.make_inputs(cfg), synth.make_cotangents(cfg)
    O, Sf, h = run_fwd(params_of(cfg), x, need_bwd=True)
    g, _ = run_bwd(params_of(cfg), h, ct)
    parts = [np.load(os.path.join(tmp_path, f"rank{r}.npz")) for r in range(2)]
    assert np.array_equal(np.concatenate([p["O"] for p in parts]), O)
    assert np.array_equal(np.concatenate([p["dq"] for p in parts]), g["dq"])
    wg = shard.pack_weight_grads(g)
    for p in parts:   # summed in a different order than the single-GPU reduction: equal to fp32 rounding
        assert np.max(np.abs(p["wg"] - wg)) <= 1e-5 * max(np.max(np.abs(wg)), 1e-30)
