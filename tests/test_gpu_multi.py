"""Tests that need TWO visible GPUs (skipped on a one-GPU box): the one-slab-per-rank driver over NCCL
(slabs of slices on several GPUs) and contexts on a device that is not the current one."""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest

from paper_1809_09725_b200 import synth

pytestmark = pytest.mark.gpu
ROOT = Path(__file__).resolve().parents[1]
CASE = synth.CONFIGS[3].scaled(cfg=41, n=72, nd=80, nz=9, n_angles=60, n_half_rot=3, m=8, n_objects=6)
N_IT = 6
TAU, SIGMA = 0.012, 0.011


def _need_two_gpus():
    import torch
    if not torch.cuda.is_available() or torch.cuda.device_count() < 2:
        pytest.skip("needs 2 CUDA devices")
    return torch


def _rank_worker(rank, world, port, out_dir):
    """One rank = one z-slab on its own GPU; the two halo slices travel as NCCL point-to-point pairs (slabs.iterate_rank)."""
    sys.path.insert(0, str(ROOT))
    import torch
    import torch.distributed as dist
    from paper_1809_09725_b200 import slabs
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    c = CASE
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    g = synth.sinogram(c).numpy().astype(np.float32)
    R = slabs.RankSlab(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m, phi, rank, world, device=rank,
                       lambda1=c.lambda1, lambda2=c.lambda2)
    R.ctx.set_data(torch.as_tensor(g[R.z0:R.z1], device=f"cuda:{rank}").contiguous())
    R.ctx.set_steps(TAU, SIGMA)
    R.ctx.reset()
    slabs.iterate_rank(R, rank, world, N_IT)
    R.ctx.sync()
    np.savez(Path(out_dir) / f"rank{rank}.npz", z0=R.z0, z1=R.z1, **{k: v.cpu().numpy() for k, v in R.st.items() if k != "g"})
    dist.barrier()
    dist.destroy_process_group()


def test_rank_slabs_over_nccl_match_whole_volume(tmp_path):
    torch = _need_two_gpus()
    import torch.multiprocessing as mp
    from paper_1809_09725_b200 import binding
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    procs = [ctx.Process(target=_rank_worker, args=(r, 2, port, str(tmp_path))) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(timeout=600)
        assert p.exitcode == 0
    c = CASE
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    g = synth.sinogram(c).numpy().astype(np.float32)
    whole = binding.Context.from_config(c, phi=phi)
    whole.set_data(torch.as_tensor(g, device="cuda")); whole.set_steps(TAU, SIGMA); whole.reset(); whole.iterate(N_IT); whole.sync()
    sw = {k: v.cpu().numpy() for k, v in whole.state().items()}
    for r in range(2):
        d = np.load(tmp_path / f"rank{r}.npz")
        z0, z1 = int(d["z0"]), int(d["z1"])
        for k in ("f", "ft", "h1"):
            ref = sw[k][z0:z1]
            assert np.linalg.norm(d[k] - ref) <= 1e-5 * np.linalg.norm(ref), (r, k)
        ref = sw["h2"][:, z0:z1]
        assert np.linalg.norm(d["h2"] - ref) <= 1e-5 * np.linalg.norm(ref), (r, "h2")
    whole.close()


def test_context_on_a_device_that_is_not_current():
    """Every entry point selects the context's device for its duration and restores the caller's (include/cp4d.h)."""
    torch = _need_two_gpus()
    from paper_1809_09725_b200 import binding
    c = CASE
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    torch.cuda.set_device(0)
    ctx1 = binding.Context.from_config(c, phi=phi, device=1)
    assert torch.cuda.current_device() == 0
    ctx0 = binding.Context.from_config(c, phi=phi, device=0)
    f = torch.randn(ctx0.primal_shape, generator=torch.Generator().manual_seed(1)).to(torch.float32)
    g0 = ctx0.forward(f.to("cuda:0"))
    g1 = ctx1.forward(f.to("cuda:1"))              # current device is 0: the call must run on device 1
    ctx1.sync()
    assert torch.cuda.current_device() == 0
    assert g1.device.index == 1
    a, b = g0.cpu().numpy(), g1.cpu().numpy()
    assert np.linalg.norm(a - b) <= 1e-5 * np.linalg.norm(a)      # RED order may differ between launches
    ctx0.close(); ctx1.close()
