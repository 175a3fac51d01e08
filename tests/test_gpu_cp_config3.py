"""Multi-iteration Chambolle-Pock parity at config 3 IN FULL (512 x 512 x 32, 1440 angles, m = 16; Fig. 2).

SURVEY 8(c) P-plan row 3: the fast oracle (same C code, OpenMP over outputs, bitwise equal to one thread) does one whole
config-3 iteration in about 10 s on the GPU box's host cores, so the real thing is affordable: the config's own synthetic data,
tau = sigma = 0.95 / L with L from the power iteration, zero start, and the iterates compared after the run -- not one
teacher-forced step.  Three checks, each with the oracle running inside the test (no cached expected values):

  1. power iteration (L97, L147, L170; R8): the oracle's start vector is handed to the GPU (cp4d_norm_start), so the
     comparison is iterate for iterate, rel 1e-4 on L -- not "both converged";
  2. 20 iterations with the config's lambda1 = 1e-3, lambda2 = 1 (C18): rel-L2 <= 1e-3 on f, ft, h1, h2, clamp fraction reported;
  3. a short run with a lambda1 that puts half of the 4-vectors on each branch of max(1, |q|/lambda1) at iteration 2 (C18).
     lambda1 is chosen with the oracle alone: after iteration 1 (where h2 stays 0 whatever lambda1 is) it is the median of
     |sigma grad ft|, i.e. of the |q| of iteration 2; the run goes on to iteration 4 (clamp fraction reported).
"""
import time

import numpy as np
import pytest

from paper_1809_09725_b200 import synth

pytestmark = pytest.mark.gpu
TOL_CP = 1e-3


def rel(a, b):
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    return float(np.linalg.norm(a.ravel() - b.ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


@pytest.fixture(scope="module")
def fast_oracle(oracle):
    oracle.set_threads(oracle.max_threads())
    yield oracle
    oracle.set_threads(1)


@pytest.fixture(scope="module")
def problem(torch_cuda, fast_oracle):
    from paper_1809_09725_b200 import binding
    c = synth.CONFIGS[3]
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    P = fast_oracle.Problem.from_config(c, phi=phi)
    with torch_cuda.cuda.stream(torch_cuda.cuda.Stream()):      # a capturable stream: cp4d_iterate replays its CUDA graph, as in bench.py
        ctx = binding.Context.from_config(c, phi=phi)
    g32 = synth.sinogram(c).numpy().astype(np.float32)          # both sides get the fp32-rounded data
    yield c, P, ctx, g32
    ctx.close()


def _dev(torch, a):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float32), device="cuda")


N_POWER = 10


def test_power_iteration_same_start(torch_cuda, problem):
    c, P, ctx, _ = problem
    x0 = synth.rng(c.cfg, 3).standard_normal(P.primal_shape).astype(np.float32)
    t0 = time.perf_counter()
    L_ref, _ = P.power(x0.astype(np.float64), N_POWER, folded=True)
    t_or = time.perf_counter() - t0
    xd = _dev(torch_cuda, x0)
    L = ctx.norm_start(xd, N_POWER)
    print(f"config 3 power iteration, {N_POWER} steps from the same start: oracle {L_ref:.6f} ({t_or:.0f} s), gpu {L:.6f}")
    assert abs(L - L_ref) <= 1e-4 * L_ref
    # the step sizes bench.py uses rest on 30 steps from the library's own start vector: the estimates grow with the step count
    # (power iteration on a symmetric positive semi-definite operator) and tau sigma L^2 = 0.9025 leaves 5 % for what is missing
    L30 = ctx.norm(30, seed=3)
    L60 = ctx.norm(60, seed=3)
    print(f"gpu norm(30) {L30:.6f}, norm(60) {L60:.6f}")
    assert L30 >= L * (1 - 1e-4) and L60 >= L30 * (1 - 1e-6)
    assert (0.95 / L30) ** 2 * L60 ** 2 < 0.95          # tau sigma |K|^2 < 1 with margin (L60 stands in for |K|)


def test_cp_20_iterations_config_lambda(torch_cuda, problem):
    torch = torch_cuda
    c, P, ctx, g32 = problem
    n_it = 20
    L = ctx.norm(30, seed=3)
    ts = float(np.float32(0.95 / L))
    gd = _dev(torch, g32)                                          # kept alive until the sync: the context runs on its own stream
    ctx.set_data(gd); ctx.set_steps(ts, ts); ctx.reset(); ctx.iterate(n_it); ctx.sync()
    assert ctx.graph_replays() > 0, ctx.graph_note()
    st = P.zero_state()
    t0 = time.perf_counter()
    ncl = P.cp(g32.astype(np.float64), st, ts, ts, n_it, folded=True)
    t_or = time.perf_counter() - t0
    s = ctx.state()
    errs = {k: rel(s[k].cpu().numpy(), st[k]) for k in ("f", "ft", "h1", "h2")}
    print(f"config 3, {n_it} CP iterations, lambda1 = {c.lambda1}: clamp fraction {ncl / (P.V):.3f}, rel-L2 {errs}, oracle {t_or:.0f} s")
    for k, e in errs.items():
        assert e <= TOL_CP, (k, e)
    assert np.isfinite(st["f"]).all() and np.linalg.norm(st["f"]) > 0


def test_cp_mixed_branches(torch_cuda, problem):
    torch = torch_cuda
    c, P, ctx, g32 = problem
    L = ctx.norm(30, seed=3)
    ts = float(np.float32(0.95 / L))
    g64 = g32.astype(np.float64)
    st = P.zero_state()
    P.cp(g64, st, ts, ts, 1, folded=True)                         # iteration 1: q = 0, h2 stays 0 for every lambda1 > 0
    assert not st["h2"].any()
    q = ts * P.grad(st["ft"])
    lam = float(np.float32(np.median(np.sqrt((q ** 2).sum(0)))))   # half of the 4-vectors of iteration 2 exceed it
    del q
    assert lam > 0
    P.lambda1 = lam
    ctx2 = type(ctx).from_config(c, phi=synth.basis_table(c.basis, c.m, c.n_angles), lambda1=lam)
    gd = _dev(torch, g32)
    ctx2.set_data(gd); ctx2.set_steps(ts, ts); ctx2.reset()
    done = 1
    try:
        for more, want_mixed in ((1, True), (2, False)):            # after iteration 2 (half / half by construction), then after 4
            ncl = P.cp(g64, st, ts, ts, more, folded=True)
            done += more
            ctx2.iterate(done if done == 2 else more); ctx2.sync()
            frac = ncl / P.V
            s = ctx2.state()
            errs = {k: rel(s[k].cpu().numpy(), st[k]) for k in ("f", "ft", "h1", "h2")}
            print(f"config 3, {done} CP iterations, lambda1 = {lam:.4g}: clamp fraction at the last step {frac:.3f}, rel-L2 {errs}")
            if want_mixed:
                assert 0.3 < frac < 0.7
            for k, e in errs.items():
                assert e <= TOL_CP, (k, e)
    finally:
        P.lambda1 = c.lambda1
        ctx2.close()
