"""Pins of the fp64 oracle (oracle/cp4d_ref.c) against what the paper and the mathematics fix.

None of these calls the CUDA path.  Pin numbering P1..P8 follows SURVEY.md section 8(c) / DESIGN.md.
"""
import numpy as np
import pytest

from oracle import dense
from paper_1809_09725_b200 import synth


def tiny(oracle, n=8, nz=2, nd=8, n_angles=16, n_half_rot=2, m=2, lambda1=0.05, lambda2=1.5, seed=0):
    phi = np.random.default_rng(seed).standard_normal((m, n_angles))
    return oracle.Problem(n, nz, nd, n_angles, n_half_rot, m, phi, lambda1, lambda2)


# ---------------------------------------------------------------- P1: static Joseph matrix (O1)
@pytest.mark.parametrize("n,nd", [(8, 8), (9, 12), (16, 11), (32, 32)])
def test_p1_ray_stepping_equals_closed_form(oracle, n, nd):
    """Ray-stepping forward (C) == dense hat-function matrix typed in numpy, incl. 0, 45, 90, 135 deg."""
    n_angles = 8
    P = oracle.Problem(n, 1, nd, n_angles, 1, 1, np.ones((1, n_angles)))
    f = np.random.default_rng(1).standard_normal(P.primal_shape)
    g = P.forward(f)
    for k in range(n_angles):
        A = dense.joseph_matrix(n, nd, k * np.pi / n_angles)
        np.testing.assert_allclose(g[0, k], A @ f.ravel(), atol=1e-12)
        np.testing.assert_allclose(P.dense_A(k), A, atol=1e-13)
        assert (A > 0).sum(axis=0).max() <= 2          # each (voxel, angle) touches at most 2 bins


def test_p1_axis_angles_are_column_and_row_sums(oracle):
    n = 16
    P = oracle.Problem(n, 1, n, 2, 1, 1, np.ones((1, 2)))     # theta = 0, pi/2
    f = np.random.default_rng(2).standard_normal((n, n))
    g = P.forward(f.reshape(P.primal_shape))
    np.testing.assert_allclose(g[0, 0], f.sum(axis=0), atol=1e-12)   # theta=0: integrate over y
    np.testing.assert_allclose(g[0, 1], f.sum(axis=1), atol=1e-12)   # theta=pi/2: integrate over x


# ---------------------------------------------------------------- P2: K1 / K1^T vs brute force
def test_p2_dense_bruteforce_forward_and_adjoint(oracle):
    P = tiny(oracle)
    K = dense.dense_K1(P.n, P.nz, P.nd, P.n_angles, P.n_half_rot, P.m, P.phi)
    rng = np.random.default_rng(3)
    f, g = rng.standard_normal(P.primal_shape), rng.standard_normal(P.sino_shape)
    np.testing.assert_allclose(P.forward(f).ravel(), K @ f.ravel(), atol=1e-12)
    np.testing.assert_allclose(P.adjoint(g).ravel(), K.T @ g.ravel(), atol=1e-12)
    np.testing.assert_allclose(P.forward(f, folded=True).ravel(), K @ f.ravel(), atol=1e-12)
    np.testing.assert_allclose(P.adjoint(g, folded=True).ravel(), K.T @ g.ravel(), atol=1e-12)


@pytest.mark.parametrize("cfg,kw", [(1, {}), (2, dict(n=48, nd=48, nz=3, n_angles=96)), (4, dict(n=24, nd=30, nz=2, n_angles=40))])
def test_p2_adjoint_dot_product(oracle, cfg, kw):
    c = synth.CONFIGS[cfg].scaled(**kw)
    P = oracle.Problem.from_config(c)
    f, g = synth.test_vectors(c)
    Kf, Ktg = P.forward(f), P.adjoint(g)
    lhs, rhs = np.vdot(Kf, g), np.vdot(f, Ktg)
    assert abs(lhs - rhs) <= 1e-12 * np.linalg.norm(Kf) * np.linalg.norm(g)
    Kf2, Ktg2 = P.forward(f, folded=True), P.adjoint(g, folded=True)
    assert np.linalg.norm(Kf2 - Kf) <= 1e-13 * np.linalg.norm(Kf)
    assert np.linalg.norm(Ktg2 - Ktg) <= 1e-13 * np.linalg.norm(Ktg)


def test_sampled_entry_points_equal_full(oracle):
    c = synth.CONFIGS[1].scaled(nz=2)
    P = oracle.Problem.from_config(c)
    f, g = synth.test_vectors(c)
    rng = np.random.default_rng(5)
    zkb = np.stack([rng.integers(0, c.nz, 64), rng.integers(0, c.n_angles, 64), rng.integers(0, c.nd, 64)], 1)
    zyx = np.stack([rng.integers(0, c.nz, 64), rng.integers(0, c.n, 64), rng.integers(0, c.n, 64)], 1)
    Kf, Ktg = P.forward(f), P.adjoint(g)
    np.testing.assert_array_equal(P.forward_rays(f, zkb), Kf[zkb[:, 0], zkb[:, 1], zkb[:, 2]])
    np.testing.assert_array_equal(P.adjoint_voxels(g, zyx), Ktg[zyx[:, 0], zyx[:, 1], zyx[:, 2]])


def test_thread_count_does_not_change_bits(oracle):
    c = synth.CONFIGS[1].scaled(nz=3)
    P = oracle.Problem.from_config(c)
    f, g = synth.test_vectors(c)
    a1, b1, c1 = P.forward(f), P.adjoint(g), P.adjoint(g, folded=True)
    oracle.set_threads(4)
    try:
        np.testing.assert_array_equal(P.forward(f), a1)
        np.testing.assert_array_equal(P.adjoint(g), b1)
        np.testing.assert_array_equal(P.adjoint(g, folded=True), c1)
    finally:
        oracle.set_threads(1)


# ---------------------------------------------------------------- P3: closed-form Radon transforms
def _radon_errors(oracle, n, kind):
    n_angles = 12
    P = oracle.Problem(n, 1, n, n_angles, 1, 1, np.ones((1, n_angles)))
    x = np.arange(n) - (n - 1) / 2.0
    X, Y = np.meshgrid(x, x, indexing="xy")
    s = np.arange(n) - (n - 1) / 2.0
    if kind == "gauss":
        sig = n / 10.0
        img = np.exp(-(X ** 2 + Y ** 2) / (2 * sig ** 2))
        exact = sig * np.sqrt(2 * np.pi) * np.exp(-s ** 2 / (2 * sig ** 2))
    else:
        r = 0.3 * n
        img = (X ** 2 + Y ** 2 <= r ** 2).astype(float)
        exact = 2 * np.sqrt(np.maximum(0.0, r ** 2 - s ** 2))
    g = P.forward(img.reshape(P.primal_shape))[0]
    return np.linalg.norm(g - exact[None]) / np.linalg.norm(np.repeat(exact[None], n_angles, 0))


def test_p3_gaussian_radon_second_order(oracle):
    e = [_radon_errors(oracle, n, "gauss") for n in (32, 64, 128)]
    assert e[1] < 2e-3
    for a, b in zip(e, e[1:]):
        assert 3.7 < a / b < 4.3          # exact 2nd-order convergence of the Joseph sum


def test_p3_disk_radon(oracle):
    e = [_radon_errors(oracle, n, "disk") for n in (32, 64, 128)]
    assert e[1] < 2.5e-2 and e[0] > e[1] > e[2]


# ---------------------------------------------------------------- P4: pi-periodicity fold (A8)
def test_p4_pi_symmetry_of_static_matrix(oracle):
    P = oracle.Problem(12, 1, 15, 40, 4, 1, np.ones((1, 40)))
    n0 = 10
    for k in range(n0):
        for q in range(1, 4):
            A0, Aq = P.dense_A(k), P.dense_A(k + q * n0)
            np.testing.assert_allclose(Aq, A0[::-1] if q % 2 else A0, atol=1e-13)


# ---------------------------------------------------------------- P5: proxes
def test_p5_prox_f1_optimality(oracle):
    """h' minimises <h',g> + |h'|^2/2 + |h-h'|^2/(2 sigma)  <=>  g + h' + (h'-h)/sigma = 0."""
    P = tiny(oracle)
    rng = np.random.default_rng(7)
    h, kf, g = (rng.standard_normal(P.sino_shape) for _ in range(3))
    sigma = 0.37
    hp = P.prox_f1(h, kf, g, sigma)
    arg = h + sigma * kf          # the prox argument of step 3
    np.testing.assert_allclose(g + hp + (hp - arg) / sigma, 0, atol=1e-13)


def test_p5_prox_f2_moreau_and_projection(oracle):
    """prox_{sigma F*}(q) = q - sigma * prox_{F/sigma}(q/sigma), F = lambda1*|.|_2 pointwise (vector soft threshold)."""
    P = tiny(oracle, lambda1=0.8)
    rng = np.random.default_rng(8)
    h2 = rng.standard_normal((4,) + P.primal_shape)
    gr = rng.standard_normal((4,) + P.primal_shape)
    sigma = 0.6
    out, ncl = P.prox_f2(h2, gr, sigma)
    q = h2 + sigma * gr
    nq = np.sqrt((q ** 2).sum(0))
    shrink = np.maximum(0.0, 1.0 - (P.lambda1 / sigma) / np.maximum(nq / sigma, 1e-300)) * (q / sigma)
    np.testing.assert_allclose(out, q - sigma * shrink, atol=1e-13)
    no = np.sqrt((out ** 2).sum(0))
    assert no.max() <= P.lambda1 * (1 + 1e-14)
    inside = nq <= P.lambda1
    assert 0 < inside.sum() < inside.size and ncl == (~inside).sum()
    np.testing.assert_array_equal(out[:, inside], q[:, inside])
    # direction preserved
    np.testing.assert_allclose(out * nq, q * no, atol=1e-13)


# ---------------------------------------------------------------- P6: grad / div / norms
def test_p6_grad_is_dense_forward_difference_and_div_is_minus_transpose(oracle):
    P = tiny(oracle, n=5, nz=3, m=4, lambda2=2.0)
    K2 = dense.dense_K2(P.n, P.nz, P.m, P.lambda2)
    rng = np.random.default_rng(9)
    f, p = rng.standard_normal(P.primal_shape), rng.standard_normal((4,) + P.primal_shape)
    np.testing.assert_allclose(P.grad(f).ravel(), K2 @ f.ravel(), atol=1e-13)
    np.testing.assert_allclose(P.div(p).ravel(), -(K2.T @ p.ravel()), atol=1e-13)
    np.testing.assert_array_equal(P.grad(np.full(P.primal_shape, 3.25)), 0.0)
    assert abs(np.vdot(P.grad(f), p) + np.vdot(f, P.div(p))) < 1e-12


def test_p6_axis_of_length_one_contributes_nothing(oracle):
    c = synth.CONFIGS[1]
    P = oracle.Problem.from_config(c)
    f = synth.test_vectors(c)[0]
    assert np.all(P.grad(f)[2] == 0)


@pytest.mark.parametrize("n,nz,m,lam2", [(5, 3, 6, 2.0), (8, 1, 4, 1.0)])
def test_p6_norm_K2_closed_form(oracle, n, nz, m, lam2):
    """||K2||^2 = sum_a w_a^2 (2 - 2 cos(pi (n_a-1)/n_a)): largest eigenvalue of path-graph Laplacians."""
    P = tiny(oracle, n=n, nz=nz, m=m, lambda2=lam2)
    lap = lambda k: 0.0 if k == 1 else 2 - 2 * np.cos(np.pi * (k - 1) / k)
    closed = 2 * lap(n) + lap(nz) + lam2 ** 2 * lap(m)
    sv = np.linalg.svd(dense.dense_K2(n, nz, m, lam2), compute_uv=False)[0]
    assert abs(sv ** 2 - closed) < 1e-10
    x0 = np.random.default_rng(10).standard_normal(P.primal_shape)
    Ls = [P.power(x0, k, use_k1=False)[0] for k in (5, 50, 3000)]
    assert Ls[0] <= Ls[1] <= Ls[2] <= np.sqrt(closed) * (1 + 1e-12)     # converges from below
    assert abs(Ls[2] ** 2 - closed) < 1e-3 * closed
    assert closed < 4 * (3 + lam2 ** 2)


def test_p6_power_iteration_vs_dense_svd(oracle):
    P = tiny(oracle)
    K = np.vstack([dense.dense_K1(P.n, P.nz, P.nd, P.n_angles, P.n_half_rot, P.m, P.phi),
                   dense.dense_K2(P.n, P.nz, P.m, P.lambda2)])
    smax = np.linalg.svd(K, compute_uv=False)[0]
    x0 = np.random.default_rng(11).standard_normal(P.primal_shape)
    L60, L, = P.power(x0, 60)[0], P.power(x0, 4000)[0]      # random table: top singular values are close
    assert L60 <= L <= smax * (1 + 1e-12) and abs(L - smax) <= 1e-6 * smax


def test_p6_config1_norm_value(oracle):
    """||K|| of config 1 (geometry + 4-term Fourier table, lambda2 = 1) against the dense SVD."""
    c = synth.CONFIGS[1]
    P = oracle.Problem.from_config(c)
    K = np.vstack([dense.dense_K1(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m, P.phi), dense.dense_K2(c.n, c.nz, c.m, 1.0)])
    smax = np.linalg.svd(K, compute_uv=False)[0]
    L, _ = P.power(synth.rng(1, 3).standard_normal(P.primal_shape), 30)
    assert abs(L - smax) < 1e-6 * smax
    golden = float(open(__file__.replace("test_oracle_pins.py", "golden/config1_norm.txt")).read().split()[0])
    assert abs(L - golden) < 1e-9 * golden


# ---------------------------------------------------------------- P7: the CP loop
def _cp_setup(oracle, lambda1, seed=12, **kw):
    P = tiny(oracle, lambda1=lambda1, **kw)
    K1 = dense.dense_K1(P.n, P.nz, P.nd, P.n_angles, P.n_half_rot, P.m, P.phi)
    K2 = dense.dense_K2(P.n, P.nz, P.m, P.lambda2)
    g = np.random.default_rng(seed).standard_normal(P.sino_shape)
    L = np.linalg.svd(np.vstack([K1, K2]), compute_uv=False)[0]
    return P, K1, K2, g, 0.95 / L


@pytest.mark.parametrize("theta", [1.0, 0.5, 0.0])
def test_p7_cp_step_matches_dense_algebra(oracle, theta):
    """Three iterations of Fig. 2 written with dense matrices (steps 3-6 verbatim) == the C loop, for the over-relaxation
    theta = 1 (R7) and for theta = 0.5, 0 (theta in [0,1])."""
    P, K1, K2, g, ts = _cp_setup(oracle, 0.3)
    st = P.zero_state()
    f = np.zeros(P.V); ft = f.copy(); h1 = np.zeros(P.S); h2 = np.zeros(4 * P.V)
    for it in range(3):
        P.cp(g, st, ts, ts, 1, theta=theta)
        h1 = (h1 + ts * (K1 @ ft) - ts * g.ravel()) / (1 + ts)                       # step 3
        q = (h2 + ts * (K2 @ ft)).reshape(4, -1)                                     # step 4
        h2 = (q / np.maximum(1.0, np.sqrt((q ** 2).sum(0)) / P.lambda1)).ravel()
        fn = f - ts * (K1.T @ h1) - ts * (K2.T @ h2)                                 # step 5 (div = -K2^T)
        ft = fn + theta * (fn - f)                                                   # step 6
        f = fn
        np.testing.assert_allclose(st["f"].ravel(), f, atol=1e-12)
        np.testing.assert_allclose(st["ft"].ravel(), ft, atol=1e-12)
        np.testing.assert_allclose(st["h1"].ravel(), h1, atol=1e-12)
        np.testing.assert_allclose(st["h2"].ravel(), h2, atol=1e-12)


def test_p7_lambda1_zero_is_least_squares(oracle):
    P, K1, K2, g, ts = _cp_setup(oracle, 0.0)
    st = P.zero_state()
    P.cp(g, st, ts, ts, 1000)
    f = st["f"].ravel()
    assert np.all(st["h2"] == 0)
    U, s, Vt = np.linalg.svd(K1)
    null = Vt[(s > 1e-10 * s[0]).sum():]
    assert np.linalg.norm(null @ f) <= 1e-12 * max(1.0, np.linalg.norm(f))           # f in range(K1^T)
    res = np.linalg.norm(K1.T @ (K1 @ f - g.ravel())) / np.linalg.norm(K1.T @ g.ravel())
    assert res < 1e-2
    P.cp(g, st, ts, ts, 4000)
    f = st["f"].ravel()
    res2 = np.linalg.norm(K1.T @ (K1 @ f - g.ravel())) / np.linalg.norm(K1.T @ g.ravel())
    assert res2 < 0.5 * res


def test_p7_kkt_fejer_and_stationarity(oracle):
    P, K1, K2, g, ts = _cp_setup(oracle, 0.3)
    K = np.vstack([K1, K2])
    # long run -> (f*, h*)
    star = P.zero_state()
    P.cp(g, star, ts, ts, 60000)
    fs, hs = star["f"].ravel(), np.concatenate([star["h1"].ravel(), star["h2"].ravel()])
    kkt0 = np.linalg.norm(K1.T @ g.ravel())
    # (ii) KKT at the limit
    assert np.linalg.norm(K.T @ hs) < 1e-6 * kkt0
    np.testing.assert_allclose(star["h1"].ravel(), K1 @ fs - g.ravel(), atol=1e-6 * np.linalg.norm(g))
    h2 = star["h2"].reshape(4, -1)
    gf = (K2 @ fs).reshape(4, -1)
    assert np.sqrt((h2 ** 2).sum(0)).max() <= P.lambda1 * (1 + 1e-12)
    ng = np.sqrt((gf ** 2).sum(0))
    act = ng > 1e-6 * ng.max()
    assert act.any()
    np.testing.assert_allclose((h2 * gf).sum(0)[act], P.lambda1 * ng[act], rtol=1e-4)
    # (iv) a stationary point stays stationary
    nxt = {k: v.copy() for k, v in star.items()}
    P.cp(g, nxt, ts, ts, 1)
    assert np.linalg.norm(nxt["f"] - star["f"]) < 1e-9 * np.linalg.norm(star["f"])
    # (iii) Fejer monotonicity in the CP metric |f-f*|^2/tau - 2<K(f-f*),h-h*> + |h-h*|^2/sigma, and KKT residual decay
    st = P.zero_state()
    prev, kkt = np.inf, []
    for n in range(200):
        P.cp(g, st, ts, ts, 1)
        df = st["f"].ravel() - fs
        dh = np.concatenate([st["h1"].ravel(), st["h2"].ravel()]) - hs
        d = df @ df / ts - 2 * (K @ df) @ dh + dh @ dh / ts
        assert d <= prev * (1 + 1e-9) + 1e-12
        prev = d
        kkt.append(np.linalg.norm(K.T @ np.concatenate([st["h1"].ravel(), st["h2"].ravel()])))
    assert kkt[-1] < 0.1 * kkt[0]


# ---------------------------------------------------------------- P8: basis tables (inputs)
@pytest.mark.parametrize("m,na", [(4, 128), (8, 720), (16, 1440)])
def test_p8_fourier_table_orthogonality(m, na):
    phi = synth.basis_table("fourier", m, na)
    np.testing.assert_allclose(phi @ phi.T / na, np.diag([1.0] + [0.5] * (m - 1)), atol=1e-13)
    t = np.arange(na) / na
    if m == 4:   # the four functions config 1 lists
        np.testing.assert_allclose(phi, [np.ones(na), np.cos(2 * np.pi * t), np.sin(2 * np.pi * t), np.cos(4 * np.pi * t)], atol=1e-15)


def test_p8_bspline_partition_of_unity():
    phi = synth.basis_table("bspline", 16, 3000)
    np.testing.assert_allclose(phi.sum(0), 1.0, atol=1e-13)
    assert phi.min() >= 0 and (phi > 0).sum(0).max() <= 4


def test_synthetic_data_is_exact_radon_of_disks(oracle):
    """Noise-free config-1 data (analytic disk integrals) vs the oracle projecting a rasterised static phantom:
    pins the geometry conventions (bin centre, angle direction) shared by generator and oracle."""
    c = synth.CONFIGS[1].scaled(n=128, nd=128, n_angles=32, n_half_rot=1)
    p = synth.phantom_params(c)
    p0 = dict(p); p0["vel"] = p["vel"] * 0
    import paper_1809_09725_b200.synth as S
    orig = S.phantom_params
    S.phantom_params = lambda cc: p0
    try:
        g = S.sinogram(c, noise=False).numpy()
    finally:
        S.phantom_params = orig
    x = np.arange(c.n) - (c.n - 1) / 2.0
    X, Y = np.meshgrid(x, x, indexing="xy")
    img = np.zeros((c.n, c.n))
    for o in range(c.n_objects):
        img += p0["rho"][o] * ((X - p0["c0"][o, 0]) ** 2 + (Y - p0["c0"][o, 1]) ** 2 <= p0["A0"][o] ** 2)
    P = oracle.Problem(c.n, 1, c.nd, c.n_angles, 1, 1, np.ones((1, c.n_angles)))
    gp = P.forward(img.reshape(P.primal_shape))
    assert np.linalg.norm(gp - g) / np.linalg.norm(g) < 3e-2


# ---------------------------------------------------------------- P9: the paper's frame discretisation (L214-L237)
def _frame_problem(oracle, n_frames, basis="fourier", m=4, n=8, nz=2, nd=8, n_angles=16, n_half_rot=2, lambda1=0.05, lambda2=1.5):
    phi = synth.basis_table(basis, m, n_angles)
    return oracle.FrameProblem(n, nz, nd, n_angles, n_half_rot, m, phi, n_frames, lambda1=lambda1, lambda2=lambda2), phi


def test_p9_frame_operator_is_dense_K1_times_analysis(oracle):
    """K1' = K1 (I (x) Psi) with Psi[j,q] = phi_j(t_q) typed here from the definition t_q = (q N_theta/N_t)/N_theta (Eq. 11)."""
    F, phi = _frame_problem(oracle, 8)
    P = F.coef
    t_q = (np.arange(8) * (P.n_angles // 8)) / P.n_angles
    psi = np.stack([np.ones(8), np.cos(2 * np.pi * t_q), np.sin(2 * np.pi * t_q), np.cos(4 * np.pi * t_q)])   # config-1 basis list
    K = dense.dense_K1(P.n, P.nz, P.nd, P.n_angles, P.n_half_rot, P.m, P.phi) @ np.kron(np.eye(P.nz * P.n * P.n), psi)
    rng = np.random.default_rng(5)
    u, g = rng.standard_normal(F.primal_shape), rng.standard_normal(F.sino_shape)
    np.testing.assert_allclose(F.forward(u).ravel(), K @ u.ravel(), atol=1e-12)
    np.testing.assert_allclose(F.adjoint(g).ravel(), K.T @ g.ravel(), atol=1e-12)
    assert abs(np.vdot(F.forward(u, folded=True), g) - np.vdot(u, F.adjoint(g, folded=True))) <= 1e-12 * np.linalg.norm(u) * np.linalg.norm(g) * 50


def test_p9_cardinal_basis_with_Nt_equal_M_is_the_coefficient_model(oracle):
    """With the box basis and N_t = M, phi_j(t_q) = delta_jq: frames are coefficients (C1) and the two CP loops coincide."""
    F, phi = _frame_problem(oracle, 4, basis="box")
    np.testing.assert_array_equal(F.psi, np.eye(4))
    P = F.coef
    g = np.random.default_rng(6).standard_normal(P.sino_shape)
    sa, sb = P.zero_state(), F.zero_state()
    P.cp(g, sa, 0.01, 0.02, 6)
    F.cp(g, sb, 0.01, 0.02, 6)
    for k in ("f", "ft", "h1", "h2"):
        np.testing.assert_allclose(sb[k], sa[k], rtol=0, atol=1e-13)


def test_p9_frame_cp_step_matches_dense_algebra(oracle):
    F, phi = _frame_problem(oracle, 8)
    P = F.coef
    K1 = dense.dense_K1(P.n, P.nz, P.nd, P.n_angles, P.n_half_rot, P.m, P.phi) @ np.kron(np.eye(P.nz * P.n * P.n), F.psi)
    K2 = dense.dense_K2(P.n, P.nz, 8, 1.5)
    rng = np.random.default_rng(7)
    st = dict(f=rng.standard_normal(F.primal_shape), ft=rng.standard_normal(F.primal_shape),
              h1=rng.standard_normal(F.sino_shape), h2=0.05 * rng.standard_normal((4,) + F.primal_shape))
    g = rng.standard_normal(F.sino_shape)
    tau, sigma, lam1 = 0.02, 0.03, 0.05
    h1 = (st["h1"].ravel() + sigma * (K1 @ st["ft"].ravel() - g.ravel())) / (1 + sigma)
    q = (st["h2"].ravel() + sigma * (K2 @ st["ft"].ravel())).reshape(4, -1)
    h2 = q / np.maximum(1.0, np.sqrt((q ** 2).sum(0)) / lam1)
    f = st["f"].ravel() - tau * (K1.T @ h1) - tau * (K2.T @ h2.ravel())
    ft = 2 * f - st["f"].ravel()
    F.cp(g, st, tau, sigma, 1)
    np.testing.assert_allclose(st["h1"].ravel(), h1, atol=1e-12)
    np.testing.assert_allclose(st["h2"].reshape(4, -1), h2, atol=1e-12)
    np.testing.assert_allclose(st["f"].ravel(), f, atol=1e-12)
    np.testing.assert_allclose(st["ft"].ravel(), ft, atol=1e-12)


# ---------------------------------------------------------------- P10: static FBP per half-rotation (L243, L257-L259)
def test_p10_shepp_logan_kernel_properties(oracle):
    h = oracle.shepp_logan_kernel(4097)
    assert h[4096] == pytest.approx(2.0 / np.pi ** 2)                   # h[0]
    assert np.all(np.delete(h, 4096) < 0)                                # negative side lobes
    assert abs(h.sum()) < 1e-4                                           # sum over Z of -2/(pi^2 (4n^2-1)) = 0: no DC gain
    # its transfer function is the band-limited ramp |sin(w/2)| / pi  (= |xi| for xi = w / 2 pi -> 0)
    n = np.arange(-4096, 4097)
    for w in (0.05, 0.5, 1.0, 2.0, 3.0):
        assert np.sum(h * np.cos(w * n)) == pytest.approx(abs(np.sin(w / 2.0)) / np.pi, rel=1e-3, abs=1e-5)


def test_p10_fbp_reconstructs_a_disk(oracle):
    """Exact Radon data of a centred disk (closed form 2 sqrt(r^2 - s^2)), two half-rotations: every half-rotation's FBP is the
    disk: ~1 inside, ~0 outside (Joseph backprojector + unit-spacing filter: a few per cent)."""
    n = nd = 64
    na, npi, r = 180, 2, 18.0
    s = np.arange(nd) - (nd - 1) / 2.0
    row = 2.0 * np.sqrt(np.maximum(0.0, r * r - s * s))
    g = np.broadcast_to(row, (1, na, nd)).copy()
    rec = oracle.fbp_half_rotations(n, 1, nd, na, npi, g)
    assert rec.shape == (1, n, n, npi)
    x = np.arange(n) - (n - 1) / 2.0
    rho = np.hypot(*np.meshgrid(x, x))
    for q in range(npi):
        img = rec[0, :, :, q]
        assert abs(img[rho < r - 3].mean() - 1.0) < 0.02
        assert np.abs(img[rho < r - 3] - 1.0).max() < 0.08
        assert np.abs(img[(rho > r + 3) & (rho < 30)]).max() < 0.08
    np.testing.assert_allclose(rec[..., 0], rec[..., 1], atol=1e-9)     # symmetric data: the bin flip changes nothing


def test_p10_fbp_follows_a_disk_that_moves_between_half_rotations(oracle):
    """An OFF-CENTRE disk that jumps to another place at every half-rotation ("time frames 3, 4 ... by using
    projections from the intervals [3 pi, 4 pi) and [4 pi, 5 pi)").  Data: exact chord lengths at the TRUE angle theta_k = k pi/n0
    (>= pi from the second half-rotation on, so the detector coordinate is mirrored there, L202).  Plane q of the FBP must show
    the disk where it was during half-rotation q and nothing where it was during the others: a half-rotation assigned to the
    wrong plane, or an odd one backprojected without the flip, lands the disk at the wrong place (the positions are chosen so
    that no two of them, nor their mirror images, overlap)."""
    n = nd = 64
    n0, npi, r = 120, 3, 6.0
    na = n0 * npi
    centres = [(12.0, 5.0), (-9.0, 11.0), (4.0, -14.0)]
    s = np.arange(nd) - (nd - 1) / 2.0
    g = np.zeros((1, na, nd))
    for k in range(na):
        th = k * np.pi / n0
        cx, cy = centres[k // n0]
        g[0, k] = 2.0 * np.sqrt(np.maximum(0.0, r * r - (s - cx * np.cos(th) - cy * np.sin(th)) ** 2))
    rec = oracle.fbp_half_rotations(n, 1, nd, na, npi, g)
    x = np.arange(n) - (n - 1) / 2.0
    X, Y = np.meshgrid(x, x, indexing="xy")
    for q in range(npi):
        img = rec[0, :, :, q]
        for p, (cx, cy) in enumerate(centres):
            inside = np.hypot(X - cx, Y - cy) < r - 2.5
            mirrored = np.hypot(X + cx, Y + cy) < r - 2.5        # where a missing flip would put it
            if p == q:
                assert abs(img[inside].mean() - 1.0) < 0.05, (q, p, img[inside].mean())
                assert abs(img[mirrored].mean()) < 0.1
            else:
                assert abs(img[inside].mean()) < 0.1, (q, p, img[inside].mean())
        # centre of mass of the clearly positive part sits at the disk of this half-rotation
        w = np.where(img > 0.5, img, 0.0)
        assert abs((w * X).sum() / w.sum() - centres[q][0]) < 0.5 and abs((w * Y).sum() / w.sum() - centres[q][1]) < 0.5
