"""The one-pass step of cp4d_iterate (include/cp4d.h: cp4d_workspace_bytes_fused; Fig. 2,
L147-L168, steps 4-6 in one pass over the volume): a context created on the larger workspace must give the iterates of the
two-kernel path -- against the fp64 oracle within north_star's tolerance, and against the two-kernel context to rounding --
for every tile shape (Q = m / 4 from 1 to 8 float4 per voxel, ragged tile edges, z chunks with a recomputed slice below,
one slice), with the double-buffered arrays swapping roles under graph replay and odd iteration counts."""
import numpy as np
import pytest

from paper_1809_09725_b200 import synth

pytestmark = pytest.mark.gpu


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


@pytest.fixture(scope="module")
def fast_oracle(oracle):
    oracle.set_threads(oracle.max_threads())
    yield oracle
    oracle.set_threads(1)


CASES = {
    # Q = 4, tiles of 16 x 6 voxels: 75 = 4 * 16 + 11 = 12 * 6 + 3 (ragged in x and y)
    "q4_ragged": (synth.CONFIGS[3].scaled(cfg=41, n=75, nd=90, nz=5, n_angles=60, n_half_rot=2, m=16, n_objects=3), 0),
    "q1": (synth.CONFIGS[2].scaled(cfg=42, n=50, nd=61, nz=3, n_angles=48, n_half_rot=2, m=4), 0),
    # few tiles: the launcher splits z into chunks, each of which recomputes the prox of the slice below it
    "q8_zchunks": (synth.CONFIGS[3].scaled(cfg=43, n=40, nd=50, nz=9, n_angles=40, n_half_rot=2, m=32, n_objects=3), 0),
    "q3_zchunks": (synth.CONFIGS[3].scaled(cfg=44, n=33, nd=40, nz=17, n_angles=36, n_half_rot=3, m=12, n_objects=3), 0),
    "frames8": (synth.CONFIGS[2].scaled(cfg=45, n=50, nd=61, nz=3, n_angles=96, n_half_rot=2, m=4), 8),
    "one_slice": (synth.CONFIGS[2].scaled(cfg=46, n=64, nd=70, nz=1, n_angles=48, n_half_rot=2, m=8), 0),
}


def _run(torch, c, nf, fused, its, theta=1.0, warm=False):
    from paper_1809_09725_b200 import binding
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    with torch.cuda.stream(torch.cuda.Stream()):           # a capturable stream: cp4d_iterate replays its graph
        ctx = binding.Context.from_config(c, phi=phi, n_frames=nf, fused=fused, theta=theta)
        try:
            assert ctx.fused_step_in_use() == fused
            gen = torch.Generator(device="cuda")
            gen.manual_seed(5)
            truth = torch.randn(ctx.primal_shape, device="cuda", generator=gen)
            data = ctx.forward(truth)
            L = ctx.norm(8, 1)
            ctx.set_data(data); ctx.set_steps(0.95 / L, 0.95 / L)
            # warm: a non-zero initial guess (f = ft = f0), so that the first prox already sees a gradient
            ctx.reset(torch.randn(ctx.primal_shape, device="cuda", generator=gen) if warm else None)
            for n in its:
                ctx.iterate(n)
            ctx.sync()
            st = {k: v.cpu().numpy().astype(np.float64) for k, v in ctx.state().items()}
            return st, ctx.graph_replays(), ctx.launch_count()
        finally:
            ctx.close()


@pytest.mark.parametrize("case", sorted(CASES))
@pytest.mark.parametrize("its", [(1,), (2,), (5,), (3, 4, 1)])
def test_fused_step_matches_two_kernel_path(torch_cuda, case, its):
    c, nf = CASES[case]
    a, ra, _ = _run(torch_cuda, c, nf, False, its)
    b, rb, _ = _run(torch_cuda, c, nf, True, its)
    for k in ("f", "ft", "h1", "h2"):
        assert np.isfinite(b[k]).all()
        # same arithmetic per element; the projectors' atomic additions are ordered differently from run to run
        assert rel(b[k], a[k]) <= 2e-6, (k, rel(b[k], a[k]))
    assert np.linalg.norm(b["f"]) > 0 and (sum(its) < 2 or np.linalg.norm(b["h2"]) > 0)      # (h2 stays 0 in the first iteration from zero)
    # the two-kernel path replays one iteration per graph launch, the one-pass step two (the copies are back in their roles);
    # a call that finds the copies swapped launches one iteration directly first
    want_a = sum(n for n in its if n >= 2)
    want_b, flip = 0, 0
    for n in its:
        if n >= 2:
            want_b += (n - flip) // 2
            flip = (n - flip) % 2
        else:
            flip ^= n & 1
    assert (ra, rb) == (want_a, want_b)


@pytest.mark.parametrize("case", ["q4_ragged", "q3_zchunks"])
def test_fused_step_first_iteration_dual_is_bit_exact(torch_cuda, case):
    """After ONE iteration from the same non-zero initial guess h2 = proj(sigma K2 f0) on both paths: the one-pass kernel's prox
    (own voxels, and the values it stores are the ones its divergence used) must reproduce k_grad<1>'s bit for bit."""
    c, nf = CASES[case]
    a, _, _ = _run(torch_cuda, c, nf, False, (1,), warm=True)
    b, _, _ = _run(torch_cuda, c, nf, True, (1,), warm=True)
    assert np.linalg.norm(a["h2"]) > 0
    assert np.array_equal(a["h2"], b["h2"])
    for k in ("f", "ft"):
        assert rel(b[k], a[k]) <= 2e-6


@pytest.mark.parametrize("theta", [1.0, 0.5])
def test_fused_step_against_oracle(torch_cuda, fast_oracle, theta):
    """Six iterations of Fig. 2 from the same data: the one-pass context against the fp64 oracle, state by
    state, within north_star's 1e-3 (relative L2) on all four arrays, as tests/test_gpu_parity.py asks of the two-kernel path."""
    torch = torch_cuda
    from paper_1809_09725_b200 import binding
    c, _ = CASES["q4_ragged"]
    c = c.scaled(lambda1=0.004)
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    P = fast_oracle.Problem.from_config(c, phi=phi)
    r = synth.rng(c.cfg, 11)
    g = r.standard_normal(P.sino_shape).astype(np.float32)
    tau = sigma = 0.012
    st = P.zero_state()
    P.cp(g.astype(np.float64), st, tau, sigma, 6, theta=theta, folded=True)
    with torch.cuda.stream(torch.cuda.Stream()):
        ctx = binding.Context.from_config(c, phi=phi, fused=True, theta=theta)
        try:
            assert ctx.fused_step_in_use()
            ctx.set_data(torch.as_tensor(g, device="cuda")); ctx.set_steps(tau, sigma); ctx.reset(None)
            ctx.iterate(6); ctx.sync()
            got = {k: v.cpu().numpy().astype(np.float64) for k, v in ctx.state().items()}
        finally:
            ctx.close()
    for k in ("f", "ft", "h1", "h2"):
        assert rel(got[k], st[k]) <= 1e-3, (k, rel(got[k], st[k]))


def test_fused_step_needs_the_larger_workspace(torch_cuda):
    """The one-pass step is chosen by the workspace the caller provides: cp4d_workspace_bytes_fused = cp4d_workspace_bytes plus
    second copies of h2[4] and ft; a z-slab context never takes it; the state pointers follow the swap."""
    torch = torch_cuda
    from paper_1809_09725_b200 import binding
    c, _ = CASES["q1"]
    a = binding.workspace_bytes(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m)
    b = binding.workspace_bytes(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m, fused=True)
    V = c.nz * c.n * c.n * c.m
    assert 20 * V <= b - a <= 20 * V + 512
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    slab = binding.Context.from_config(c, phi=phi, z_open=2, fused=True)
    assert not slab.fused_step_in_use()
    slab.close()
    with torch.cuda.stream(torch.cuda.Stream()):
        ctx = binding.Context.from_config(c, phi=phi, fused=True)
        try:
            data = ctx.forward(ctx.empty_primal().normal_())
            ctx.set_data(data); ctx.set_steps(0.01, 0.01); ctx.reset(None)
            p0 = {k: v.data_ptr() for k, v in ctx.state().items()}
            ctx.iterate(1)
            p1 = {k: v.data_ptr() for k, v in ctx.state().items()}
            ctx.iterate(1)
            p2 = {k: v.data_ptr() for k, v in ctx.state().items()}
            assert p1["ft"] != p0["ft"] and p1["h2"] != p0["h2"] and p2 == p0
            assert all(p1[k] == p0[k] for k in ("f", "h1", "g"))
            # the profile names the one-pass kernel, and neither of the two it replaces
            ctx.profile_begin(); ctx.iterate(2)
            prof = ctx.profile_end()
            assert prof["prox_update"][1] == 2 and "prox_f2" not in prof and "update" not in prof
        finally:
            ctx.close()
