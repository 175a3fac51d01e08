"""z-slab contexts (cp4d_params.z_open, the *_slab / cp4d_step_* calls) against the
whole-volume context and the oracle: the decomposition must not change the result."""
import numpy as np
import pytest

from paper_1809_09725_b200 import synth

pytestmark = pytest.mark.gpu


def rel(a, b):
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1809_09725_b200 import build
    build.build_lib()
    return torch


CASE = synth.CONFIGS[2].scaled(cfg=41, n=45, nd=50, nz=7, n_angles=36, n_half_rot=3, m=8, lambda1=0.003, lambda2=0.7)


def dev(torch, a):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float32), device="cuda")


@pytest.mark.parametrize("n_slabs", [2, 3, 7])
def test_grad_div_slabs_bit_exact(torch_cuda, n_slabs):
    from paper_1809_09725_b200 import binding, slabs
    torch = torch_cuda
    c = CASE
    whole = binding.Context.from_config(c)
    S = slabs.SlabSolver.from_config(c, n_slabs=n_slabs)
    r = synth.rng(c.cfg, 1)
    f = dev(torch, r.standard_normal(whole.primal_shape))
    p = dev(torch, r.standard_normal((4,) + whole.primal_shape))
    g_ref, d_ref = whole.grad(f), whole.div(p)
    g_s = torch.cat(S.grad(S.split(f)), dim=1)
    d_s = torch.cat(S.div(S.split(p)), dim=0)
    assert torch.equal(g_s, g_ref) and torch.equal(d_s, d_ref)      # same arithmetic per element: bit for bit
    # the z-coupling is real: a slab without its halos differs at the interfaces
    z1 = S.ranges[0][1]
    closed = binding.Context.from_config(c.scaled(nz=z1))
    assert not torch.equal(closed.grad(S.split(f)[0])[2], g_ref[2, :z1])
    for x in (whole, closed):
        x.close()
    S.close()


@pytest.mark.parametrize("n_slabs", [2, 3])
def test_slab_solver_matches_whole_volume_and_oracle(torch_cuda, oracle, n_slabs):
    from paper_1809_09725_b200 import binding, slabs
    torch = torch_cuda
    c = CASE
    oracle.set_threads(oracle.max_threads())
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    g = synth.sinogram(c).numpy().astype(np.float32)
    whole = binding.Context.from_config(c, phi=phi)
    S = slabs.SlabSolver.from_config(c, phi=phi, n_slabs=n_slabs)
    L = whole.norm(30, seed=5)
    Ls = S.norm(30, seed=5)
    assert abs(Ls - L) <= 5e-4 * L                       # two random starts of the same power iteration
    ts = float(np.float32(0.95 / L))
    for x in (whole, S):
        x.set_data(dev(torch, g)); x.set_steps(ts, ts); x.reset(); x.iterate(12); x.sync()
    sw = whole.state()
    for k in ("f", "ft", "h1", "h2"):
        assert rel(S.gather(k).cpu().numpy(), sw[k].cpu().numpy()) <= 1e-5, k     # atomics: summation order may differ
    P = oracle.Problem.from_config(c, phi=phi)
    st = P.zero_state()
    ncl = P.cp(g.astype(np.float64), st, ts, ts, 12, folded=True)
    assert 0.02 < ncl / P.V < 0.98
    assert rel(S.get_f().cpu().numpy(), st["f"]) <= 1e-3 and rel(S.gather("h2").cpu().numpy(), st["h2"]) <= 1e-3
    oracle.set_threads(1)
    whole.close(); S.close()


@pytest.mark.parametrize("slab_nz,depth", [(2, 2), (3, 3), (7, 1)])
def test_streamed_solver_matches_in_core(torch_cuda, slab_nz, depth):
    """State in pinned host memory, slabs of slab_nz slices (ragged last slab) through `depth` device contexts."""
    from paper_1809_09725_b200 import binding, slabs
    torch = torch_cuda
    c = CASE
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    g = synth.sinogram(c).numpy().astype(np.float32)
    whole = binding.Context.from_config(c, phi=phi)
    whole.set_data(dev(torch, g)); whole.set_steps(0.012, 0.011); whole.reset(); whole.iterate(9); whole.sync()
    sw = whole.state()
    T = slabs.StreamedSolver(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m, phi, slab_nz=slab_nz, depth=depth,
                             lambda1=c.lambda1, lambda2=c.lambda2)
    T.set_data(g); T.set_steps(0.012, 0.011); T.reset(); T.iterate(5); T.iterate(4)
    f = T.get_f()
    assert rel(f.numpy(), sw["f"].cpu().numpy()) <= 1e-5
    assert rel(T.ft.numpy(), sw["ft"].cpu().numpy()) <= 1e-5
    assert rel(T.h2.numpy(), sw["h2"].cpu().numpy()) <= 1e-5
    assert rel(T.h1.numpy(), sw["h1"].cpu().numpy()) <= 1e-5
    n_sl = (c.nz + slab_nz - 1) // slab_nz
    assert T.bytes_h2d == 9 * (c.nz * (6 * c.n * c.n * c.m + 2 * c.n_angles * c.nd) + (n_sl - 1) * c.n * c.n * c.m) * 4
    T.close(); whole.close()


@pytest.mark.parametrize("slab_nz,block,iters", [(2, 2, 9), (3, 4, 8), (1, 3, 7)])
def test_streamed_solver_temporal_blocking(torch_cuda, slab_nz, block, iters):
    """block = k: windows of slab_nz + 2k slices iterated k times as closed volumes, cores written to the second host copy."""
    from paper_1809_09725_b200 import binding, slabs
    torch = torch_cuda
    c = CASE
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    g = synth.sinogram(c).numpy().astype(np.float32)
    whole = binding.Context.from_config(c, phi=phi)
    whole.set_data(dev(torch, g)); whole.set_steps(0.012, 0.011); whole.reset(); whole.iterate(iters); whole.sync()
    sw = whole.state()
    T = slabs.StreamedSolver(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m, phi, slab_nz=slab_nz, depth=2, block=block,
                             lambda1=c.lambda1, lambda2=c.lambda2)
    T.set_data(g); T.set_steps(0.012, 0.011); T.reset(); T.iterate(iters)       # iters is not a multiple of block: a short last sweep
    T.get_f()
    for k, v in (("f", T.f), ("ft", T.ft), ("h2", T.h2), ("h1", T.h1)):
        assert rel(v.numpy(), sw[k].cpu().numpy()) <= 1e-5, k
    sweeps = -(-iters // block)
    n_sl = (c.nz + slab_nz - 1) // slab_nz
    assert T.bytes_h2d == sweeps * n_sl * T.win_nz * (6 * c.n * c.n * c.m + 2 * c.n_angles * c.nd) * 4
    assert sum(x.graph_replays() for x in T._ctx.values()) > 0                   # the windows run cp4d_iterate's graph path
    T.close(); whole.close()


@pytest.mark.parametrize("n_frames", [4, 12])
def test_slabs_in_frame_mode(torch_cuda, n_frames):
    """Frame mode (N_t <= M collapsed into the projector table, N_t > M through k_mix) cut into 3 slabs, all-resident and streamed."""
    from paper_1809_09725_b200 import binding, slabs
    torch = torch_cuda
    c = CASE
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    g = synth.sinogram(c).numpy().astype(np.float32)
    whole = binding.Context.from_config(c, phi=phi, n_frames=n_frames)
    S = slabs.SlabSolver.from_config(c, phi=phi, n_slabs=3, n_frames=n_frames)
    T = slabs.StreamedSolver(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m, phi, slab_nz=3, n_frames=n_frames, block=2,
                             lambda1=c.lambda1, lambda2=c.lambda2)
    for x in (whole, S):
        x.set_data(dev(torch, g)); x.set_steps(0.01, 0.01); x.reset(); x.iterate(6); x.sync()
    T.set_data(g); T.set_steps(0.01, 0.01); T.reset(); T.iterate(6); T.get_f()
    sw = whole.state()
    assert sw["f"].shape[-1] == n_frames and float(sw["h2"].abs().max()) > 0
    for k in ("f", "ft", "h1", "h2"):
        assert rel(S.gather(k).cpu().numpy(), sw[k].cpu().numpy()) <= 1e-5, k
        assert rel(getattr(T, k).numpy(), sw[k].cpu().numpy()) <= 1e-5, k
    whole.close(); S.close(); T.close()


def test_slab_context_call_rules(torch_cuda):
    from paper_1809_09725_b200 import binding
    torch = torch_cuda
    c = CASE.scaled(nz=3)
    mid = binding.Context.from_config(c, z_open=3)
    f, p = mid.empty_primal().normal_(), mid.empty_dual().normal_()
    one = f[0].clone()
    for call in (lambda: mid.grad(f), lambda: mid.div(p), lambda: mid.iterate(2), lambda: mid.norm(2), lambda: mid.objective()):
        with pytest.raises(binding.Cp4dError) as e:
            call()
        assert e.value.code == binding.ESTATE
    for call in (lambda: mid.grad_slab(f, None), lambda: mid.div_slab(p, None)):       # a missing halo on an interior face
        with pytest.raises(binding.Cp4dError) as e:
            call()
        assert e.value.code == binding.EINVAL
    mid.grad_slab(f, one); mid.div_slab(p, one)
    mid.set_z_open(0)
    with pytest.raises(binding.Cp4dError):                                              # a halo on a closed face
        mid.grad_slab(f, one)
    assert torch.equal(mid.grad_slab(f), mid.grad(f))
    with pytest.raises(binding.Cp4dError):
        mid.set_z_open(4)
    mid.close()
