"""cp4d_forward_static (include/cp4d.h): the forward operator with the projector's scratch in the library's file-scope
__device__ array instead of the workspace -- for callers that cannot provide scratch at call time.  Its output is checked
against the existing path (cp4d_forward, same kernels) on two calls in a row with different inputs (the array keeps the last
call's contents: a missing zero-fill would show in the second call), in both projector modes, and against the fp64 oracle;
a problem beyond CP4D_STATIC_SCRATCH_BYTES is refused with CP4D_ETOOLARGE.  Collected last (file name) on purpose."""
import numpy as np
import pytest

from paper_1809_09725_b200 import synth

pytestmark = pytest.mark.gpu

TOL_OP = 1e-4          # BASELINE.json north_star: relative L2 per operator against the oracle
TOL_SAME = 1e-5        # against cp4d_forward: same kernels, only the order of the projector's atomic additions differs


def rel(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1809_09725_b200 import build
    build.build_lib()
    return torch


# spans several tiles with a ragged tail, four-angle groups in the tensor kernel (90 base angles), 6.3 MB of partial sums
CASE = synth.CONFIGS[3].scaled(cfg=31, n=75, nd=90, nz=5, n_angles=180, n_half_rot=2, m=16, n_objects=5)


@pytest.mark.parametrize("mode", ["fp32", "tensor"])
def test_forward_static_matches_forward_twice(torch_cuda, oracle, mode):
    torch = torch_cuda
    from paper_1809_09725_b200 import binding
    c = CASE
    assert c.nz * c.n_theta0 * c.nd * c.m * 4 <= binding.STATIC_SCRATCH_BYTES
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    ctx = binding.Context.from_config(c, phi=phi)
    try:
        ctx.set_projector_mode(mode)
        assert ctx.projector_mode_in_use()[0] == mode
        rng = np.random.default_rng(7)
        f1 = torch.as_tensor(rng.standard_normal(ctx.primal_shape).astype(np.float32), device="cuda")
        f2 = torch.as_tensor((3.0 * rng.standard_normal(ctx.primal_shape) + 1.0).astype(np.float32), device="cuda")
        want1, want2 = ctx.forward(f1).cpu().numpy(), ctx.forward(f2).cpu().numpy()
        got1 = ctx.forward_static(f1).cpu().numpy()          # two calls in a row on the shared array
        got2 = ctx.forward_static(f2).cpu().numpy()
        got1b = ctx.forward_static(f1).cpu().numpy()         # and back: nothing of call 2 is left in it
        assert np.isfinite(got1).all() and np.isfinite(got2).all()
        assert rel(got1, want1) <= TOL_SAME
        assert rel(got2, want2) <= TOL_SAME
        assert rel(got1b, want1) <= TOL_SAME
        assert rel(want1, want2) > 0.5                       # the two calls really differ
        # and against the oracle, as the existing path is checked
        P = oracle.Problem.from_config(c, phi=phi)
        ref2 = P.forward(f2.cpu().numpy().astype(np.float64), folded=True)
        assert rel(got2, ref2) <= TOL_OP
    finally:
        ctx.close()


@pytest.mark.parametrize("nt", [8, 4])
def test_forward_static_in_frame_mode(torch_cuda, nt):
    """Frame mode: N_t = 8 > M = 4 keeps the analysis step in front of the projector (cp4d_forward_static runs it too);
    N_t = 4 <= M collapses to a coefficient-mode problem.  Against cp4d_forward, two calls in a row."""
    torch = torch_cuda
    from paper_1809_09725_b200 import binding
    c = synth.CONFIGS[2].scaled(cfg=33, n=50, nd=61, nz=3, n_angles=96, n_half_rot=2, m=4)
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    ctx = binding.Context.from_config(c, phi=phi, n_frames=nt)
    try:
        f1, f2 = ctx.empty_primal().normal_(), ctx.empty_primal().normal_()
        want1, want2 = ctx.forward(f1).cpu().numpy(), ctx.forward(f2).cpu().numpy()
        got1, got2 = ctx.forward_static(f1).cpu().numpy(), ctx.forward_static(f2).cpu().numpy()
        assert rel(got1, want1) <= TOL_SAME and rel(got2, want2) <= TOL_SAME
        assert rel(want1, want2) > 0.5
    finally:
        ctx.close()


def test_forward_static_refuses_what_does_not_fit(torch_cuda):
    torch = torch_cuda
    from paper_1809_09725_b200 import binding
    c = synth.CONFIGS[3].scaled(cfg=32, n=64, nd=256, nz=9, n_angles=360, n_half_rot=1, m=16, n_objects=2)
    assert c.nz * c.n_theta0 * c.nd * c.m * 4 > binding.STATIC_SCRATCH_BYTES
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    ctx = binding.Context.from_config(c, phi=phi)
    try:
        f = ctx.empty_primal().normal_()
        g = ctx.empty_sino().fill_(-7.0)
        with pytest.raises(binding.Cp4dError) as ei:
            ctx.forward_static(f, out=g)
        assert ei.value.code == binding.ETOOLARGE
        assert "CP4D_STATIC_SCRATCH_BYTES" in str(ei.value)
        torch.cuda.synchronize()
        assert bool((g == -7.0).all())                      # nothing was launched
        ctx.forward(f, out=g)                               # the existing path takes the same problem
        assert np.isfinite(g.cpu().numpy()).all()
    finally:
        ctx.close()
