"""Parity of the CUDA path (through the C ABI, via the ctypes binding) against the fp64 oracle, element by element
on the same seeded inputs.  Tolerances are BASELINE.json north_star's: relative L2 error <= 1e-4 per operator (fp32)
and <= 1e-3 on f after the CP iterations."""
import numpy as np
import pytest

from paper_1809_09725_b200 import synth

pytestmark = pytest.mark.gpu

TOL_OP = 1e-4
TOL_CP = 1e-3


def rel(a, b):
    a = np.asarray(a, dtype=np.float64)
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


def dev(torch, a):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float32), device="cuda")


# shapes: the two configs the oracle runs in full + ragged / odd cases spanning several tiles and a ragged tail
CASES = {
    "cfg1": synth.CONFIGS[1],
    "cfg2": synth.CONFIGS[2],
    "ragged": synth.CONFIGS[2].scaled(cfg=12, n=45, nd=50, nz=3, n_angles=35, n_half_rot=5, m=12, lambda2=0.7),
    "wide_det": synth.CONFIGS[4].scaled(cfg=14, n=40, nd=75, nz=2, n_angles=36, n_half_rot=3, m=8),
    "narrow_det_m32": synth.CONFIGS[2].scaled(cfg=15, n=70, nd=33, nz=1, n_angles=24, n_half_rot=2, m=32),
    "one_angle_per_pi": synth.CONFIGS[1].scaled(cfg=16, n=33, nd=33, nz=2, n_angles=6, n_half_rot=6, m=4),
    # m = 16: the 8-lanes-per-ray forward kernel and two coefficient groups in the backprojector, on ragged tiles
    "ragged_m16": synth.CONFIGS[3].scaled(cfg=17, n=75, nd=90, nz=3, n_angles=78, n_half_rot=3, m=16, iters=12, n_objects=5),
    # more than 512 base angles: the forward kernel reads its per-angle tables from global memory instead of the kernel parameter
    "many_angles": synth.CONFIGS[1].scaled(cfg=18, n=36, nd=41, nz=2, n_angles=530, n_half_rot=1, m=4),
    # a volume smaller than one tile and a detector wider than the scratch window
    "tiny": synth.CONFIGS[1].scaled(cfg=19, n=5, nd=9, nz=1, n_angles=14, n_half_rot=2, m=4),
    # tensor-core forward projector (forward_mma.cu): adjacent angles grouped at 1 degree (four at a time) and at the coarsest
    # spacing that still pairs (24 base angles: most strips fall back to one window per angle), 7 slices of m = 8 (3.5 batch blocks: a ragged last
    # CTA), m = 32 (two blocks per slice), m = 4 with 13 slices (4 slices per block), ragged tiles, nd != n
    "pairs_1deg_m16": synth.CONFIGS[3].scaled(cfg=22, n=100, nd=110, nz=5, n_angles=360, n_half_rot=2, m=16, n_objects=5),
    "pairs_coarse_m8": synth.CONFIGS[3].scaled(cfg=23, n=97, nd=140, nz=7, n_angles=72, n_half_rot=3, m=8, n_objects=5),
    "pairs_m32": synth.CONFIGS[2].scaled(cfg=24, n=66, nd=70, nz=3, n_angles=200, n_half_rot=2, m=32),
    "pairs_m4_z13": synth.CONFIGS[1].scaled(cfg=25, n=50, nd=47, nz=13, n_angles=90, n_half_rot=2, m=4),
    # groups of four adjacent angles (n_theta0 >= 72: 16 rays per voxel fragment where the four angles share the 8-row windows):
    # the coarsest spacing that still groups by four (many items fall back to pairs and single angles), and a base-angle count
    # that leaves groups of three and two at the ends of the passes
    "groups4_coarsest_m16": synth.CONFIGS[3].scaled(cfg=26, n=90, nd=100, nz=4, n_angles=144, n_half_rot=2, m=16, n_objects=5),
    "groups4_tail_m8": synth.CONFIGS[3].scaled(cfg=27, n=81, nd=120, nz=5, n_angles=150, n_half_rot=1, m=8, n_objects=5),
}


def make(case, fast_oracle):
    from paper_1809_09725_b200 import binding
    c = CASES[case]
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    P = fast_oracle.Problem.from_config(c, phi=phi)
    ctx = binding.Context.from_config(c, phi=phi)
    return c, P, ctx


@pytest.mark.parametrize("case", list(CASES))
def test_forward_adjoint(torch_cuda, fast_oracle, case):
    c, P, ctx = make(case, fast_oracle)
    f, g = synth.test_vectors(c)
    f32, g32 = f.astype(np.float32), g.astype(np.float32)
    ref_f, ref_a = P.forward(f32.astype(np.float64), folded=True), P.adjoint(g32.astype(np.float64), folded=True)
    # every kernel of both sides: the exact-fp32 ones and (where m allows) the tensor-core ones with split-bf16 operands, whose
    # relative error must stay well inside the tolerance (about 5e-6 measured, 1.1e-5 bound); the modes are switched
    # back and forth on one context, which also checks that the two layouts of the folded sinogram do not leak into each other
    can = c.m in (4, 8, 16, 32)
    for mode in ("tensor", "fp32", "auto"):
        ctx.set_projector_mode(mode)
        want = {"tensor": ("tensor", "tensor"), "fp32": ("fp32", "fp32"), "auto": ("fp32", "fp32")}[mode] if can else ("fp32", "fp32")
        assert ctx.projector_mode_in_use() == want      # (auto: none of these shapes fills the GPU; test_gpu_fullsize checks the switch)
        Kf = ctx.forward(dev(torch_cuda, f32)).cpu().numpy()
        Ktg = ctx.adjoint(dev(torch_cuda, g32)).cpu().numpy()
        assert rel(Kf, ref_f) <= (2e-5 if want[0] == "tensor" else TOL_OP), mode
        assert rel(Ktg, ref_a) <= (2e-5 if want[1] == "tensor" else TOL_OP), mode
    # GPU-side adjoint identity in fp32 (fp64-accumulated dots)
    lhs = ctx.dot(dev(torch_cuda, Kf), dev(torch_cuda, g32))
    rhs = ctx.dot(dev(torch_cuda, f32), dev(torch_cuda, Ktg))
    assert abs(lhs - rhs) <= 1e-5 * np.linalg.norm(Kf) * np.linalg.norm(g32)
    ctx.close()


@pytest.mark.parametrize("scale", [1e-20, 1.0, 1e20])
def test_tensor_projectors_keep_their_error_across_magnitudes(torch_cuda, fast_oracle, scale):
    """The split-bf16 operands of the tensor kernels have the exponent range of fp32: the relative error of K1 and K1^T does not
    depend on the magnitude of the data (the operators are linear, so the oracle result is scaled)."""
    from paper_1809_09725_b200 import binding
    c = CASES["groups4_coarsest_m16"]
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    P = fast_oracle.Problem.from_config(c, phi=phi)
    ctx = binding.Context.from_config(c, phi=phi)
    f, g = synth.test_vectors(c)
    f32, g32 = (f * scale).astype(np.float32), (g * scale).astype(np.float32)
    ctx.set_projector_mode("tensor")
    assert ctx.projector_mode_in_use() == ("tensor", "tensor")
    Kf = ctx.forward(dev(torch_cuda, f32)).cpu().numpy().astype(np.float64) / scale
    Ktg = ctx.adjoint(dev(torch_cuda, g32)).cpu().numpy().astype(np.float64) / scale
    assert rel(Kf, P.forward(f32.astype(np.float64) / scale, folded=True)) <= 2e-5
    assert rel(Ktg, P.adjoint(g32.astype(np.float64) / scale, folded=True)) <= 2e-5
    ctx.close()


def test_tensor_request_falls_back_beyond_its_tables(torch_cuda, fast_oracle):
    """More than 128 angle groups in a pass (here 1100 base angles in groups of four: about 138 per pass) do not fit the tensor
    forward kernel's shared-memory records: a CP4D_PROJ_TENSOR request then runs the fp32 kernels, says so, and is still right."""
    from paper_1809_09725_b200 import binding
    c = synth.CONFIGS[1].scaled(cfg=28, n=24, nd=29, nz=1, n_angles=1100, n_half_rot=1, m=4)
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    P = fast_oracle.Problem.from_config(c, phi=phi)
    ctx = binding.Context.from_config(c, phi=phi)
    f, g = synth.test_vectors(c)
    f32, g32 = f.astype(np.float32), g.astype(np.float32)
    ctx.set_projector_mode("tensor")
    assert ctx.projector_mode_in_use() == ("fp32", "fp32")
    assert rel(ctx.forward(dev(torch_cuda, f32)).cpu().numpy(), P.forward(f32.astype(np.float64), folded=True)) <= 1e-5
    assert rel(ctx.adjoint(dev(torch_cuda, g32)).cpu().numpy(), P.adjoint(g32.astype(np.float64), folded=True)) <= 1e-5
    ctx.close()


@pytest.mark.parametrize("case", list(CASES))
def test_grad_div(torch_cuda, fast_oracle, case):
    c, P, ctx = make(case, fast_oracle)
    f = synth.test_vectors(c)[0].astype(np.float32)
    p = synth.rng(c.cfg, 5).standard_normal((4,) + P.primal_shape).astype(np.float32)
    gp = ctx.grad(dev(torch_cuda, f)).cpu().numpy()
    dp = ctx.div(dev(torch_cuda, p)).cpu().numpy()
    ref_g, ref_d = P.grad(f.astype(np.float64)), P.div(p.astype(np.float64))
    assert rel(gp, ref_g) <= 1e-6 and rel(dp, ref_d) <= 1e-6
    assert np.array_equal(gp == 0, ref_g == 0) or rel(gp, ref_g) <= 1e-7      # boundary zeros in the same places
    ctx.close()


@pytest.mark.parametrize("case", ["cfg1", "ragged", "narrow_det_m32", "ragged_m16"])
def test_fused_steps(torch_cuda, fast_oracle, case):
    c, P, ctx = make(case, fast_oracle)
    r = synth.rng(c.cfg, 6)
    ft = r.standard_normal(P.primal_shape).astype(np.float32)
    f = r.standard_normal(P.primal_shape).astype(np.float32)
    g = r.standard_normal(P.sino_shape).astype(np.float32)
    h1 = r.standard_normal(P.sino_shape).astype(np.float32)
    h2 = r.standard_normal((4,) + P.primal_shape).astype(np.float32)
    sigma, tau = 0.013, 0.021
    d = lambda a: a.astype(np.float64)
    # step 3
    out = ctx.prox_f1(sigma, dev(torch_cuda, ft), dev(torch_cuda, g), dev(torch_cuda, h1)).cpu().numpy()
    assert rel(out, P.prox_f1(d(h1), P.forward(d(ft), folded=True), d(g), sigma)) <= TOL_OP
    # step 4, lambda1 chosen so both branches of max(1, .) occur
    q = d(h2) + sigma * P.grad(d(ft))
    lam = float(np.median(np.sqrt((q ** 2).sum(0))))
    ctx2 = type(ctx).from_config(c.scaled(lambda1=lam))
    ref, ncl = P.prox_f2(d(h2), P.grad(d(ft)), sigma, lambda1=float(np.float32(lam)))
    assert 0.3 < ncl / (P.V) < 0.7
    out = ctx2.prox_f2(sigma, dev(torch_cuda, ft), dev(torch_cuda, h2)).cpu().numpy()
    assert rel(out, ref) <= 1e-6
    assert np.sqrt((out.astype(np.float64) ** 2).sum(0)).max() <= lam * (1 + 1e-5)
    # lambda1 = 0: h2 = 0
    ctx0 = type(ctx).from_config(c.scaled(lambda1=0.0))
    assert float(ctx0.prox_f2(sigma, dev(torch_cuda, ft), dev(torch_cuda, h2)).abs().max()) == 0.0
    # steps 5-6
    fo, fto = ctx.primal_update(tau, dev(torch_cuda, h1), dev(torch_cuda, h2), dev(torch_cuda, f), ctx.empty_primal())
    fn = d(f) - tau * P.adjoint(d(h1), folded=True) + tau * P.div(d(h2))
    assert rel(fo.cpu().numpy(), fn) <= TOL_OP
    assert rel(fto.cpu().numpy(), fn + 1.0 * (fn - d(f))) <= TOL_OP
    for x in (ctx, ctx2, ctx0):
        x.close()


def _data(c):
    return synth.sinogram(c).numpy()


@pytest.mark.parametrize("case,lam1", [("cfg1", 1e-3), ("cfg1", "mixed"), ("cfg2", 1e-3), ("cfg2", "mixed"), ("ragged", "mixed"), ("ragged_m16", 1e-3)])
def test_cp_iterations(torch_cuda, fast_oracle, case, lam1):
    """Full CP run (config iteration counts) from zero state with the oracle's tau = sigma = 0.95/L."""
    c = CASES[case]
    g = _data(c).astype(np.float32)
    if lam1 == "mixed":      # lambda1 for which a good fraction of voxels is clamped AND a good fraction is not (C18)
        lam1 = {"cfg1": 0.02, "cfg2": 2e-4, "ragged": 0.003}[case]   # bisected with the oracle on the clamp fraction
    c = c.scaled(lambda1=float(np.float32(lam1)))
    from paper_1809_09725_b200 import binding
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    P = fast_oracle.Problem.from_config(c, phi=phi)
    ctx = binding.Context.from_config(c, phi=phi)
    L, _ = P.power(synth.rng(c.cfg, 3).standard_normal(P.primal_shape), 30, folded=True)
    ts = float(np.float32(0.95 / L))
    st = P.zero_state()
    ncl = P.cp(g.astype(np.float64), st, ts, ts, c.iters, folded=True)
    ctx.set_data(dev(torch_cuda, g))
    ctx.set_steps(ts, ts)
    ctx.reset()
    ctx.iterate(c.iters)
    ctx.sync()
    s = ctx.state()
    frac = ncl / P.V
    print(f"{case} lambda1={lam1} clamped fraction at last iteration: {frac:.3f}")
    if lam1 != 1e-3:
        assert 0.05 < frac < 0.95
    assert rel(s["f"].cpu().numpy(), st["f"]) <= TOL_CP
    assert rel(s["h1"].cpu().numpy(), st["h1"]) <= TOL_CP
    assert rel(ctx.get_f().cpu().numpy(), st["f"]) <= TOL_CP
    ctx.close()


@pytest.mark.parametrize("case", ["cfg1", "cfg2"])
def test_power_iteration(torch_cuda, fast_oracle, case):
    c, P, ctx = make(case, fast_oracle)
    # the two sides start from different random vectors (each its own generator), so both must have converged; 30 steps do
    # on configs 1-2 (R8).  (On small m = 16 problems the top of the spectrum is clustered and two starts still
    # differ by 2e-4 after 300 steps while the operators agree to 1e-7 on the iterates -- not a parity case.)
    L_ref, _ = P.power(synth.rng(c.cfg, 3).standard_normal(P.primal_shape), 30, folded=True)
    L = ctx.norm(30, seed=7)
    assert abs(L - L_ref) <= 1e-4 * L_ref
    ctx.close()


@pytest.mark.parametrize("case", ["cfg1", "cfg2", "ragged_m16", "ragged"])
def test_power_iteration_same_start(torch_cuda, fast_oracle, case):
    """cp4d_norm_start takes the oracle's start vector: the two power iterations are compared step for step (12 steps, no
    convergence needed -- the m = 16 case above that two different starts cannot settle is a parity case this way)."""
    c, P, ctx = make(case, fast_oracle)
    x0 = synth.rng(c.cfg, 3).standard_normal(P.primal_shape).astype(np.float32)
    for steps in (1, 12):
        L_ref, _ = P.power(x0.astype(np.float64), steps, folded=True)
        L = ctx.norm_start(dev(torch_cuda, x0), steps)
        assert abs(L - L_ref) <= 1e-5 * L_ref, (steps, L, L_ref)        # (SURVEY C11 asks 1e-4)
    from paper_1809_09725_b200 import binding
    with pytest.raises(binding.Cp4dError):
        ctx.norm_start(torch_cuda.zeros(P.primal_shape, device="cuda"), 3)       # a zero start vector is refused
    ctx.close()


def test_graph_note_and_device_restored(torch_cuda, fast_oracle):
    """cp4d_iterate on the legacy default stream cannot replay a graph: it must say so (cp4d_graph_note), not fall back silently;
    and no call leaves another device current than the caller's."""
    torch = torch_cuda
    from paper_1809_09725_b200 import binding
    c = CASES["cfg1"]
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    g = dev(torch, _data(c))
    cur = torch.cuda.current_device()
    with torch.cuda.stream(torch.cuda.default_stream()):
        ctx = binding.Context.from_config(c, phi=phi)
        ctx.set_data(g); ctx.set_steps(0.01, 0.01); ctx.reset(); ctx.iterate(3); ctx.sync()
        assert ctx.graph_replays() == 0 and "legacy default stream" in ctx.graph_note()
        ctx.close()
    with torch.cuda.stream(torch.cuda.Stream()):
        ctx = binding.Context.from_config(c, phi=phi)
        ctx.set_data(g); ctx.set_steps(0.01, 0.01); ctx.reset(); ctx.iterate(3); ctx.sync()
        assert ctx.graph_replays() == 3 and ctx.graph_note() == ""
        ctx.close()
    assert torch.cuda.current_device() == cur


def test_solve_host_equals_device_path(torch_cuda, fast_oracle):
    c, P, ctx = make("cfg1", fast_oracle)
    g = _data(c).astype(np.float32)
    ctx.set_steps(0.015, 0.015)
    ctx.set_data(dev(torch_cuda, g)); ctx.reset(); ctx.iterate(5)
    a = ctx.get_f().cpu()
    gh = torch_cuda.as_tensor(g).pin_memory()
    fh = torch_cuda.empty(P.primal_shape, dtype=torch_cuda.float32).pin_memory()
    ctx.solve_host(gh, 5, fh)
    assert rel(fh.numpy(), a.numpy().astype(np.float64)) <= 1e-5       # atomics: summation order may differ
    assert ctx.launch_count() > 0
    ctx.close()


@pytest.mark.parametrize("case", ["ragged", "ragged_m16"])
def test_iterate_graph_replay(torch_cuda, case):
    """On a capturable (non-default) stream cp4d_iterate captures one iteration into a CUDA graph and replays it; on the legacy
    default stream it launches kernel by kernel.  Same iterates, same launch count; new step sizes rebuild the graph."""
    from paper_1809_09725_b200 import binding
    torch = torch_cuda
    c = CASES[case].scaled(lambda1=0.003)
    g = _data(c).astype(np.float32)

    def run(ctx):
        ctx.set_data(dev(torch, g)); ctx.set_steps(0.011, 0.012); ctx.reset()
        ctx.iterate(4); ctx.iterate(3)                 # second call reuses the graph
        ctx.set_steps(0.009, 0.012); ctx.iterate(2)    # new tau: graph rebuilt
        ctx.iterate(1)                                 # single iterations are launched directly
        ctx.sync()
        s = ctx.state()
        return {k: s[k].cpu().numpy().astype(np.float64) for k in ("f", "ft", "h1", "h2")}, (ctx.launch_count(), ctx.graph_replays())

    eager = binding.Context.from_config(c)             # current stream = legacy default stream: not capturable
    a, na = run(eager)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        graph = binding.Context.from_config(c)
        b, nb = run(graph)
        graph.close()
    eager.close()
    assert na == (nb[0], 0) and nb[1] == 4 + 3 + 2
    for k in a:
        assert rel(b[k], a[k]) <= 1e-5, k               # atomics: summation order may differ


def test_relaxation_and_warm_start(torch_cuda, fast_oracle):
    """theta = 0.5 (L97: theta in [0,1]) and a non-zero initial guess through cp4d_reset(f0) (L147 'some initial guess')."""
    from paper_1809_09725_b200 import binding
    c = CASES["wide_det"].scaled(lambda1=0.01)
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    P = fast_oracle.Problem.from_config(c, phi=phi)
    ctx = binding.Context.from_config(c, phi=phi, theta=0.5)
    r = synth.rng(c.cfg, 9)
    g = r.standard_normal(P.sino_shape).astype(np.float32)
    f0 = r.standard_normal(P.primal_shape).astype(np.float32)
    st = P.zero_state()
    st["f"][:] = f0
    st["ft"][:] = f0
    P.cp(g.astype(np.float64), st, 0.004, 0.006, 7, theta=0.5, folded=True)
    ctx.set_data(dev(torch_cuda, g)); ctx.set_steps(0.004, 0.006); ctx.reset(dev(torch_cuda, f0))
    ctx.iterate(0)                                   # no-op
    assert rel(ctx.get_f().cpu().numpy(), f0) == 0.0
    ctx.iterate(3); ctx.iterate(4)                   # 3 + 4 = 7: the state machine carries over
    ctx.sync()
    s = ctx.state()
    for name in ("f", "ft", "h1", "h2"):
        assert rel(s[name].cpu().numpy(), st[name]) <= TOL_CP, name
    ctx.close()


def test_call_order_and_aliasing_errors(torch_cuda):
    from paper_1809_09725_b200 import binding
    c = CASES["cfg1"]
    ctx = binding.Context.from_config(c)
    with pytest.raises(binding.Cp4dError) as e:
        ctx.iterate(1)                               # no data, no steps
    assert e.value.code == binding.ESTATE
    f = ctx.empty_primal().zero_()
    with pytest.raises(binding.Cp4dError) as e:      # in/out aliasing is rejected
        ctx._ck(binding.lib().cp4d_grad(ctx._h, f.data_ptr(), f.data_ptr()))
    assert e.value.code == binding.EINVAL
    with pytest.raises(binding.Cp4dError) as e:
        ctx.set_steps(0.0, 1.0)
    assert e.value.code == binding.EINVAL
    ctx.close()


@pytest.mark.parametrize("case", ["cfg1", "ragged"])
def test_objective_monitor(torch_cuda, fast_oracle, case):
    """cp4d_objective against the same quantities assembled from oracle operators (Eq. 6; C19)."""
    from paper_1809_09725_b200 import binding
    c = CASES[case].scaled(lambda1=0.02)
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    P = fast_oracle.Problem.from_config(c, phi=phi)
    ctx = binding.Context.from_config(c, phi=phi)
    g = _data(c).astype(np.float32)
    ctx.set_data(dev(torch_cuda, g)); ctx.set_steps(0.01, 0.01); ctx.reset(); ctx.iterate(6); ctx.sync()
    s = {k: v.cpu().numpy().astype(np.float64) for k, v in ctx.state().items()}
    primal, dual, kkt = ctx.objective()
    gr = P.grad(s["f"])
    ref_primal = 0.5 * np.sum((P.forward(s["f"], folded=True) - g) ** 2) + float(np.float32(0.02)) * np.sqrt((gr ** 2).sum(0)).sum()
    ref_dual = -0.5 * np.sum(s["h1"] ** 2) - np.sum(s["h1"] * g)
    ref_kkt = np.linalg.norm(P.adjoint(s["h1"], folded=True) - P.div(s["h2"]))
    assert abs(primal - ref_primal) <= 1e-4 * abs(ref_primal)
    assert abs(dual - ref_dual) <= 1e-5 * max(abs(ref_dual), 1e-30)
    assert abs(kkt - ref_kkt) <= 1e-4 * ref_kkt
    # the monitor leaves the state alone
    s2 = {k: v.cpu().numpy().astype(np.float64) for k, v in ctx.state().items()}
    assert all(np.array_equal(s[k], s2[k]) for k in s)
    ctx.close()


def test_long_run_converges(torch_cuda):
    """2000 iterations at config 2 with tau = sigma = 0.95/L (tau sigma L^2 < 1, L97): every iterate finite, the primal value
    and the dual residual |K1^T h1 - div h2| fall, the duality gap estimate closes, and |h2| <= lambda1 holds throughout."""
    from paper_1809_09725_b200 import binding
    torch = torch_cuda
    c = CASES["cfg2"].scaled(lambda1=2e-4)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):                       # the CUDA-graph path
        ctx = binding.Context.from_config(c)
        g = synth.sinogram(c, device="cuda").to(torch.float32).contiguous()
        ts = 0.95 / ctx.norm(30, seed=2)
        ctx.set_data(g); ctx.set_steps(ts, ts); ctx.reset()
        hist = []
        for n in (10, 90, 400, 1500):
            ctx.iterate(n)
            hist.append(ctx.objective())
            st = ctx.state()
            assert all(bool(torch.isfinite(st[k]).all()) for k in ("f", "ft", "h1", "h2"))
            assert float(torch.sqrt((st["h2"].double() ** 2).sum(0)).max()) <= 2e-4 * (1 + 1e-5)
        assert ctx.graph_replays() == 2000
        ctx.close()
    primal, dual, kkt = zip(*hist)
    assert primal[0] > primal[1] > primal[2] > primal[3] > 0
    assert kkt[0] > kkt[1] > kkt[2] > kkt[3]
    assert primal[3] - dual[3] < 0.2 * (primal[0] - dual[0])       # conditional gap (the dual constraint K^T h = 0 holds only in the limit)


@pytest.mark.parametrize("case", ["ragged", "ragged_m16", "cfg2"])
def test_fbp_half_rotations(torch_cuda, fast_oracle, case):
    """cp4d_fbp against the oracle's plain definition; then as the initial guess of a frame-mode run."""
    c, P, ctx = make(case, fast_oracle)
    g = synth.rng(c.cfg, 11).standard_normal(P.sino_shape).astype(np.float32)
    ref = fast_oracle.fbp_half_rotations(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, g.astype(np.float64))
    out = ctx.fbp(dev(torch_cuda, g)).cpu().numpy()
    q4 = (c.n_half_rot + 3) // 4 * 4
    assert out.shape == (c.nz, c.n, c.n, q4)
    assert rel(out[..., :c.n_half_rot], ref) <= TOL_OP
    assert not out[..., c.n_half_rot:].any()
    # the call leaves the projector scratch usable: the adjoint still matches
    Ktg = ctx.adjoint(dev(torch_cuda, g)).cpu().numpy()
    assert rel(Ktg, P.adjoint(g.astype(np.float64), folded=True)) <= TOL_OP
    ctx.close()


def test_fbp_as_initial_guess_in_frame_mode(torch_cuda, fast_oracle):
    from paper_1809_09725_b200 import binding
    c = synth.CONFIGS[1].scaled(cfg=25, n=40, nd=44, nz=2, n_angles=64, n_half_rot=4, m=4, lambda1=7e-4)
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    F = fast_oracle.FrameProblem(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m, phi, 4, lambda1=c.lambda1, lambda2=c.lambda2)
    ctx = binding.Context.from_config(c, phi=phi, n_frames=4)          # N_t = N_pi: one frame per half-rotation
    g = synth.rng(c.cfg, 1).standard_normal(F.sino_shape).astype(np.float32)
    f0 = fast_oracle.fbp_half_rotations(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, g.astype(np.float64))
    st = F.zero_state()
    st["f"][:] = f0; st["ft"][:] = f0
    F.cp(g.astype(np.float64), st, 0.004, 0.004, 6, folded=True)
    f0_gpu = ctx.fbp(dev(torch_cuda, g))
    ctx.set_data(dev(torch_cuda, g)); ctx.set_steps(0.004, 0.004); ctx.reset(f0_gpu); ctx.iterate(6); ctx.sync()
    assert rel(ctx.get_f().cpu().numpy(), st["f"]) <= TOL_CP
    ctx.close()
