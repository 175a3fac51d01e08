"""Frame mode (cp4d_params.n_frames > 0): the paper's own temporal discretisation against
the oracle's FrameProblem -- operators element-wise, fused steps, a full CP run, and the cardinal-basis special case."""
import numpy as np
import pytest

from paper_1809_09725_b200 import synth

pytestmark = pytest.mark.gpu
TOL_OP, TOL_CP = 1e-4, 1e-3

CASES = {
    # (config-like shape, n_frames); lambda1 picked with the oracle so that step 4 clamps a part of the 4-vectors, not all
    "m4_nt8": (synth.CONFIGS[1].scaled(cfg=21, n=40, nd=44, nz=2, n_angles=64, n_half_rot=4, m=4, lambda1=7e-4, lambda2=0.7), 8),
    "m16_nt8": (synth.CONFIGS[3].scaled(cfg=22, n=45, nd=50, nz=3, n_angles=48, n_half_rot=3, m=16, lambda1=7e-4, lambda2=1.3), 8),
    "m8_nt12": (synth.CONFIGS[4].scaled(cfg=23, n=33, nd=40, nz=2, n_angles=36, n_half_rot=2, m=8, lambda1=0.03), 12),
}


def rel(a, b):
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def dev(torch, a):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float32), device="cuda")


def make(case, oracle):
    from paper_1809_09725_b200 import binding
    c, nt = CASES[case]
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    F = oracle.FrameProblem(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m, phi, nt, lambda1=c.lambda1, lambda2=c.lambda2)
    ctx = binding.Context.from_config(c, phi=phi, n_frames=nt)
    return c, nt, F, ctx


@pytest.mark.parametrize("case", list(CASES))
def test_frame_operators(torch_cuda, oracle, case):
    c, nt, F, ctx = make(case, oracle)
    assert ctx.primal_shape == (c.nz, c.n, c.n, nt)
    r = synth.rng(c.cfg, 2)
    u = r.standard_normal(F.primal_shape).astype(np.float32)
    g = r.standard_normal(F.sino_shape).astype(np.float32)
    p = r.standard_normal((4,) + F.primal_shape).astype(np.float32)
    d = lambda a: a.astype(np.float64)
    Ku = ctx.forward(dev(torch_cuda, u)).cpu().numpy()
    Ktg = ctx.adjoint(dev(torch_cuda, g)).cpu().numpy()
    assert rel(Ku, F.forward(d(u), folded=True)) <= TOL_OP
    assert rel(Ktg, F.adjoint(d(g), folded=True)) <= TOL_OP
    assert rel(ctx.grad(dev(torch_cuda, u)).cpu().numpy(), F.grad(d(u))) <= 1e-6
    assert rel(ctx.div(dev(torch_cuda, p)).cpu().numpy(), F.div(d(p))) <= 1e-6
    lhs = ctx.dot(dev(torch_cuda, Ku), dev(torch_cuda, g))
    rhs = ctx.dot(dev(torch_cuda, u), dev(torch_cuda, Ktg))
    assert abs(lhs - rhs) <= 1e-5 * np.linalg.norm(Ku) * np.linalg.norm(g)
    ctx.close()


@pytest.mark.parametrize("case", list(CASES))
def test_frame_cp_run(torch_cuda, oracle, case):
    c, nt, F, ctx = make(case, oracle)
    g = synth.rng(c.cfg, 1).standard_normal(F.sino_shape).astype(np.float32)
    L = ctx.norm(30, seed=5)
    ts = float(np.float32(0.95 / L))
    st = F.zero_state()
    ncl = F.cp(g.astype(np.float64), st, ts, ts, 10, folded=True)
    ctx.set_data(dev(torch_cuda, g)); ctx.set_steps(ts, ts); ctx.reset(); ctx.iterate(10); ctx.sync()
    s = ctx.state()
    for k in ("f", "ft", "h1", "h2"):
        assert rel(s[k].cpu().numpy(), st[k]) <= TOL_CP, k
    assert 0.03 < ncl / F.frames.V < 0.97, ncl / F.frames.V      # both branches of max(1, |q|/lambda1) at the last step
    primal, dual, kkt = ctx.objective()
    gr = F.grad(st["f"])
    ref_primal = 0.5 * np.sum((F.forward(st["f"], folded=True) - g) ** 2) + float(np.float32(c.lambda1)) * np.sqrt((gr ** 2).sum(0)).sum()
    assert abs(primal - ref_primal) <= 1e-3 * abs(ref_primal)
    ctx.close()


def test_cardinal_frames_equal_coefficient_mode(torch_cuda, oracle):
    """Box basis with N_t = M: Psi = I, so frame mode and coefficient mode must produce the same iterates (C1)."""
    from paper_1809_09725_b200 import binding
    c = synth.CONFIGS[1].scaled(cfg=24, n=40, nd=44, nz=2, n_angles=64, n_half_rot=4, m=8, basis="box", lambda1=0.02)
    phi = synth.basis_table("box", c.m, c.n_angles)
    g = synth.rng(c.cfg, 1).standard_normal((c.nz, c.n_angles, c.nd)).astype(np.float32)
    outs = []
    for nt in (0, 8):
        ctx = binding.Context.from_config(c, phi=phi, n_frames=nt)
        ctx.set_data(dev(torch_cuda, g)); ctx.set_steps(0.01, 0.01); ctx.reset(); ctx.iterate(8); ctx.sync()
        outs.append(ctx.get_f().cpu().numpy().astype(np.float64))
        ctx.close()
    assert rel(outs[1], outs[0]) <= 1e-5          # summation orders differ (atomics), nothing else
