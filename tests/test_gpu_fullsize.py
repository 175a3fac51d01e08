"""Full-size parity (SURVEY 8(c) P-plan, rows 3-5): configs 3, 4, 5 in the launch configuration bench.py times.

A full fp64 oracle run is infeasible at these sizes (1e13 .. 1.5e15 FMA), so parity is
  * sampled per operator: 4096 seeded rays (forward) and 4096 seeded voxels (adjoint) in slices 0, nz/2, nz-1, each
    computed one by one by the oracle (cp4d_ref_forward_rays / cp4d_ref_adjoint_voxels), rel-L2 <= 1e-4;
  * one teacher-forced Chambolle-Pock iteration (Fig. 2) from a seeded random state: the oracle
    recomputes step 3 at the sampled rays, step 4 on 66x66 in-plane windows (two true corners + centre), and steps 5-6
    at voxels inside those windows, from the GPU's own state of the previous step copied to the host.
Inputs are torch CUDA generator streams with fixed seeds (no value comes from the kernels under test).
"""
import numpy as np
import pytest

from paper_1809_09725_b200 import synth

pytestmark = pytest.mark.gpu
TOL_OP = 1e-4
NS = 4096
WSZ = 66


def rel(a, b):
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


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


def _slices(c):
    return sorted({0, c.nz // 2, c.nz - 1})


def _sub_problem(oracle, c, phi, nz, n=None, **kw):
    n = c.n if n is None else n
    return oracle.Problem(n, nz, c.nd, c.n_angles, c.n_half_rot, c.m, phi, **kw)


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_sampled_forward_adjoint(torch_cuda, fast_oracle, cfg):
    torch = torch_cuda
    from paper_1809_09725_b200 import binding
    c = synth.CONFIGS[cfg]
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    ctx = binding.Context.from_config(c, phi=phi)
    gen = torch.Generator(device="cuda").manual_seed(1000 + cfg)
    zs = _slices(c)
    P3 = _sub_problem(fast_oracle, c, phi, len(zs))
    r = synth.rng(cfg, 7)
    # ---- forward: rays sampled in (slice, angle, bin)
    f = torch.randn(ctx.primal_shape, generator=gen, device="cuda", dtype=torch.float32)
    Kf = ctx.forward(f)
    zi = r.integers(0, len(zs), NS)
    zkb_local = np.stack([zi, r.integers(0, c.n_angles, NS), r.integers(0, c.nd, NS)], 1).astype(np.int32)
    f3 = np.stack([f[z].cpu().numpy() for z in zs]).astype(np.float64)
    ref = P3.forward_rays(f3, zkb_local)
    zsel = torch.as_tensor(np.asarray(zs)[zi], device="cuda")
    pick = lambda K: K[zsel, torch.as_tensor(zkb_local[:, 1].astype(np.int64), device="cuda"),
                       torch.as_tensor(zkb_local[:, 2].astype(np.int64), device="cuda")].cpu().numpy()
    assert ctx.projector_mode_in_use() == ("tensor", "tensor")                # the kernels bench.py times (split-bf16 sparse MMA, fp32 accumulate)
    e_tensor = rel(pick(Kf), ref)
    ctx.set_projector_mode("fp32")                                  # and the exact-fp32 gather on the same rays
    e_fp32 = rel(pick(ctx.forward(f, out=Kf)), ref)
    ctx.set_projector_mode("auto")
    print(f"config {cfg}: sampled forward rel-L2 tensor {e_tensor:.2e}, fp32 {e_fp32:.2e}")
    assert e_tensor <= 2e-5 and e_fp32 <= TOL_OP
    del f3
    # ---- adjoint: voxels sampled in (slice, y, x), all m coefficients each
    g = torch.randn(ctx.sino_shape, generator=gen, device="cuda", dtype=torch.float32)
    Ktg = ctx.adjoint(g, out=f)                                   # reuse f's memory
    zyx_local = np.stack([zi, r.integers(0, c.n, NS), r.integers(0, c.n, NS)], 1).astype(np.int32)
    g3 = np.stack([g[z].cpu().numpy() for z in zs]).astype(np.float64)
    ref = P3.adjoint_voxels(g3, zyx_local)
    got = Ktg[zsel, torch.as_tensor(zyx_local[:, 1].astype(np.int64), device="cuda"),
              torch.as_tensor(zyx_local[:, 2].astype(np.int64), device="cuda")].cpu().numpy()
    assert rel(got, ref) <= 2e-5                                  # (auto mode: the tensor-core backprojector at these sizes)
    ctx.set_projector_mode("fp32")                                # the fp32 patch kernel on the same voxels
    Ktg = ctx.adjoint(g, out=Ktg)
    assert rel(Ktg[zsel, torch.as_tensor(zyx_local[:, 1].astype(np.int64), device="cuda"),
                   torch.as_tensor(zyx_local[:, 2].astype(np.int64), device="cuda")].cpu().numpy(), ref) <= 1e-5
    ctx.set_projector_mode("tensor")                              # and the tensor mode asked for explicitly
    Ktg = ctx.adjoint(g, out=Ktg)
    e_tensor = rel(Ktg[zsel, torch.as_tensor(zyx_local[:, 1].astype(np.int64), device="cuda"),
                       torch.as_tensor(zyx_local[:, 2].astype(np.int64), device="cuda")].cpu().numpy(), ref)
    ctx.set_projector_mode("auto")
    Ktg = ctx.adjoint(g, out=Ktg)
    print(f"config {cfg}: sampled adjoint rel-L2 tensor {e_tensor:.2e}")
    assert e_tensor <= 2e-5
    # ---- fp32 adjoint identity on the GPU: <K1 f, g> = <f, K1^T g> (f was overwritten, so redo it with a fresh pair)
    f2 = torch.randn(ctx.primal_shape, generator=gen, device="cuda", dtype=torch.float32)
    Kf = ctx.forward(f2, out=Kf)
    lhs, rhs = ctx.dot(Kf, g), ctx.dot(f2, Ktg)
    assert abs(lhs - rhs) <= 1e-5 * float(Kf.norm()) * float(g.norm())
    ctx.close()


def _zsub(c, z):
    """Slices around z needed for the z-differences, and z's index among them."""
    lo, hi = max(0, z - 1), min(c.nz - 1, z + 1)
    return list(range(lo, hi + 1)), z - lo


def _valid(c, o0, size):
    """Index range of a window [o0, o0+size) along an in-plane axis where grad and div do not see the window's own edge."""
    return (0 if o0 == 0 else 1), (size if o0 + size == c.n else size - 1)


@pytest.mark.parametrize("cfg,fused", [(3, False), (4, False), (5, False), (3, True), (5, True)])
def test_teacher_forced_cp_step(torch_cuda, fast_oracle, cfg, fused):
    """One iteration of Fig. 2 from a random state at full size, checked step by step on sampled rays and windows.  fused: the
    context bench.py times (workspace of cp4d_workspace_bytes_fused: steps 4-6 as the one-pass kernel)."""
    torch = torch_cuda
    from paper_1809_09725_b200 import binding
    c = synth.CONFIGS[cfg]
    lam1, lam2, sigma, tau = 1.8, 0.8, 0.05, 0.03          # lam1 ~ median |h2 + sigma grad ft|: both prox branches occur
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    ctx = binding.Context.from_config(c, phi=phi, lambda1=lam1, lambda2=lam2, fused=fused)
    assert ctx.fused_step_in_use() == fused
    gen = torch.Generator(device="cuda").manual_seed(2000 + cfg)
    st = ctx.state()
    for name in ("f", "ft", "h1", "h2", "g"):
        st[name].normal_(generator=gen)
    zs = _slices(c)
    r = synth.rng(cfg, 8)
    cpu = lambda t: t.cpu().numpy().astype(np.float64)
    # ---- old state needed by the oracle, copied before the step
    zi = r.integers(0, len(zs), NS)
    kk, bb = r.integers(0, c.n_angles, NS), r.integers(0, c.nd, NS)
    zsel = torch.as_tensor(np.asarray(zs)[zi], device="cuda")
    tk, tb = torch.as_tensor(kk, device="cuda"), torch.as_tensor(bb, device="cuda")
    h1_old, g_s = cpu(st["h1"][zsel, tk, tb]), cpu(st["g"][zsel, tk, tb])
    ft3 = np.stack([cpu(st["ft"][z]) for z in zs])
    wins = [(0, 0), (c.n - WSZ, c.n - WSZ), ((c.n - WSZ) // 2, (c.n - WSZ) // 2 + 3)]
    old = {}
    for z in zs:
        zz, _ = _zsub(c, z)
        for (y0, x0) in wins:
            sl = (slice(zz[0], zz[-1] + 1), slice(y0, y0 + WSZ), slice(x0, x0 + WSZ))
            old[(z, y0, x0)] = dict(ft=cpu(st["ft"][sl]), f=cpu(st["f"][sl]), h2=cpu(st["h2"][(slice(None),) + sl]))
    # ---- one iteration on the GPU
    ctx._ck(binding.lib().cp4d_set_data(ctx._h, st["g"].clone().data_ptr()))
    ctx.set_steps(tau, sigma)
    ctx.iterate(1)
    ctx.sync()
    st = ctx.state()                                       # (the one-pass step wrote ft and h2 to their second copies)
    # ---- step 3 at the sampled rays
    P3 = _sub_problem(fast_oracle, c, phi, len(zs))
    kf = P3.forward_rays(ft3, np.stack([zi, kk, bb], 1).astype(np.int32))
    ref_h1 = (h1_old + sigma * (kf - g_s)) / (1.0 + sigma)
    assert rel(cpu(st["h1"][zsel, tk, tb]), ref_h1) <= TOL_OP
    del ft3
    # ---- steps 4-6 on the windows
    phi1 = np.ones((c.m, 1))
    h1_new3 = np.stack([cpu(st["h1"][z]) for z in zs])
    n_clamped = n_total = 0
    for zidx, z in enumerate(zs):
        zz, zc = _zsub(c, z)
        for (y0, x0) in wins:
            o = old[(z, y0, x0)]
            Pw = fast_oracle.Problem(WSZ, len(zz), WSZ, 1, 1, c.m, phi1, lambda1=lam1, lambda2=lam2)
            (ya, yb), (xa, xb) = _valid(c, y0, WSZ), _valid(c, x0, WSZ)
            sl = (slice(zz[0], zz[-1] + 1), slice(y0, y0 + WSZ), slice(x0, x0 + WSZ))
            # step 4: slice z of the sub-volume has its true z-neighbours (or is the true first / last slice)
            ref_h2, ncl = Pw.prox_f2(o["h2"], Pw.grad(o["ft"]), sigma, lambda1=float(np.float32(lam1)))
            got_h2 = cpu(st["h2"][(slice(None),) + sl])
            assert rel(got_h2[:, zc, ya:yb, xa:xb], ref_h2[:, zc, ya:yb, xa:xb]) <= 1e-5
            n_clamped += ncl
            n_total += o["ft"].size
            # steps 5-6: f+ = f - tau K1^T h1 + tau div h2 with the GPU's own new h1, h2 (teacher forcing)
            dv = Pw.div(got_h2)[zc, ya:yb, xa:xb]
            ys, xs = np.meshgrid(np.arange(y0 + ya, y0 + yb, 7), np.arange(x0 + xa, x0 + xb, 7), indexing="ij")
            zyx = np.stack([np.full(ys.size, zidx), ys.ravel(), xs.ravel()], 1).astype(np.int32)
            bp = P3.adjoint_voxels(h1_new3, zyx).reshape(ys.shape + (c.m,))
            f_old = o["f"][zc, ya:yb:7, xa:xb:7]
            f_ref = f_old - tau * bp + tau * dv[::7, ::7]
            f_got = cpu(st["f"][z, y0 + ya:y0 + yb:7, x0 + xa:x0 + xb:7])
            ft_got = cpu(st["ft"][z, y0 + ya:y0 + yb:7, x0 + xa:x0 + xb:7])
            assert rel(f_got, f_ref) <= TOL_OP
            assert rel(ft_got, f_ref + 1.0 * (f_ref - f_old)) <= TOL_OP
    assert 0.2 < n_clamped / n_total < 0.8, (n_clamped, n_total)     # both branches of max(1, |q|/lambda1) exercised
    ctx.close()


@pytest.mark.parametrize("cfg,nt", [(3, 8), (4, 8)])
def test_sampled_frame_mode(torch_cuda, fast_oracle, cfg, nt):
    """Frame mode at full size: N_t = 8 frames, M = 16 basis functions -- the collapsed route
    (projectors carry the frames) against the oracle's K1 o A at sampled rays / voxels."""
    torch = torch_cuda
    from paper_1809_09725_b200 import binding
    c = synth.CONFIGS[cfg]
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    psi = phi[:, ::c.n_angles // nt]                                   # Psi[j,q] = phi_j(t_q), Eq. 11
    ctx = binding.Context.from_config(c, phi=phi, n_frames=nt)
    assert ctx.primal_shape == (c.nz, c.n, c.n, nt)
    gen = torch.Generator(device="cuda").manual_seed(3000 + cfg)
    zs = _slices(c)
    P3 = _sub_problem(fast_oracle, c, phi, len(zs))
    r = synth.rng(cfg, 9)
    u = torch.randn(ctx.primal_shape, generator=gen, device="cuda", dtype=torch.float32)
    Ku = ctx.forward(u)
    zi = r.integers(0, len(zs), NS)
    kk, bb = r.integers(0, c.n_angles, NS), r.integers(0, c.nd, NS)
    f3 = np.stack([u[z].cpu().numpy() for z in zs]).astype(np.float64) @ psi.T          # analysis, L231-L237
    ref = P3.forward_rays(f3, np.stack([zi, kk, bb], 1).astype(np.int32))
    zsel = torch.as_tensor(np.asarray(zs)[zi], device="cuda")
    got = Ku[zsel, torch.as_tensor(kk, device="cuda"), torch.as_tensor(bb, device="cuda")].cpu().numpy()
    assert rel(got, ref) <= TOL_OP
    del f3
    g = torch.randn(ctx.sino_shape, generator=gen, device="cuda", dtype=torch.float32)
    Ktg = ctx.adjoint(g, out=u)
    yy, xx = r.integers(0, c.n, NS), r.integers(0, c.n, NS)
    g3 = np.stack([g[z].cpu().numpy() for z in zs]).astype(np.float64)
    ref = P3.adjoint_voxels(g3, np.stack([zi, yy, xx], 1).astype(np.int32)) @ psi       # A^T after K1^T
    got = Ktg[zsel, torch.as_tensor(yy, device="cuda"), torch.as_tensor(xx, device="cuda")].cpu().numpy()
    assert rel(got, ref) <= TOL_OP
    ctx.close()
