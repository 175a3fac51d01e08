"""ctypes front end of the fp64 CPU oracle (oracle/cp4d_ref.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this module; it imports nothing from the CUDA package.  `build()` compiles the C file with gcc.
All arrays are float64 numpy, layouts as in the header of cp4d_ref.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SO = _HERE / "libcp4d_ref.so"
_lib = None


def build(force: bool = False) -> Path:
    src = _HERE / "cp4d_ref.c"
    if force or not _SO.exists() or _SO.stat().st_mtime < src.stat().st_mtime:
        tmp = _SO.with_suffix(f".tmp{os.getpid()}.so")
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-shared", "-fPIC", "-o", str(tmp), str(src), "-lm"])
        os.replace(tmp, _SO)
    return _SO


class _Prob(C.Structure):
    _fields_ = [("n", C.c_int32), ("nz", C.c_int32), ("nd", C.c_int32), ("n_angles", C.c_int32),
                ("n_half_rot", C.c_int32), ("m", C.c_int32), ("lambda1", C.c_double), ("lambda2", C.c_double),
                ("phi", C.c_void_p)]


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(str(_SO))
        _lib.cp4d_ref_power.restype = C.c_double
        _lib.cp4d_ref_cp.restype = C.c_int64
        _lib.cp4d_ref_prox_f2.restype = C.c_int64
        _lib.cp4d_ref_max_threads.restype = C.c_int
        _lib.cp4d_ref_get_threads.restype = C.c_int
    return _lib


def set_threads(t: int) -> None:
    """1 = the definition (single thread); more = the 'fast oracle' (bitwise identical results)."""
    lib().cp4d_ref_set_threads(C.c_int(int(t)))


def max_threads() -> int:
    return int(lib().cp4d_ref_max_threads())


def get_threads() -> int:
    return int(lib().cp4d_ref_get_threads())


def _p(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(C.c_void_p)


class Problem:
    """Shape + basis table + (lambda1, lambda2) of one reconstruction problem, as the oracle sees it."""

    def __init__(self, n, nz, nd, n_angles, n_half_rot, m, phi, lambda1=1e-3, lambda2=1.0):
        if n_angles % n_half_rot:
            raise ValueError("n_angles must be a multiple of n_half_rot")
        if m > 64:
            raise ValueError("oracle supports m <= 64")
        self.n, self.nz, self.nd, self.n_angles, self.n_half_rot, self.m = n, nz, nd, n_angles, n_half_rot, m
        self.phi = np.ascontiguousarray(phi, dtype=np.float64).reshape(m, n_angles)
        self.lambda1, self.lambda2 = float(lambda1), float(lambda2)
        self._c = _Prob(n, nz, nd, n_angles, n_half_rot, m, self.lambda1, self.lambda2, self.phi.ctypes.data)

    @classmethod
    def from_config(cls, c, phi=None, **kw):
        from paper_1809_09725_b200 import synth  # input generators only
        if phi is None:
            phi = synth.basis_table(c.basis, c.m, c.n_angles)
        kw.setdefault("lambda1", c.lambda1)
        kw.setdefault("lambda2", c.lambda2)
        return cls(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m, phi, **kw)

    # shapes
    @property
    def primal_shape(self):
        return (self.nz, self.n, self.n, self.m)

    @property
    def sino_shape(self):
        return (self.nz, self.n_angles, self.nd)

    @property
    def V(self):
        return self.nz * self.n * self.n * self.m

    @property
    def S(self):
        return self.nz * self.n_angles * self.nd

    def _ref(self):
        self._c.lambda1, self._c.lambda2 = self.lambda1, self.lambda2
        return C.byref(self._c)

    # operators ------------------------------------------------------------------------------
    def forward(self, f, folded=False):
        f = np.ascontiguousarray(f, dtype=np.float64)
        g = np.empty(self.sino_shape)
        (lib().cp4d_ref_forward_folded if folded else lib().cp4d_ref_forward)(self._ref(), _p(f), _p(g))
        return g

    def adjoint(self, g, folded=False):
        g = np.ascontiguousarray(g, dtype=np.float64)
        f = np.empty(self.primal_shape)
        (lib().cp4d_ref_adjoint_folded if folded else lib().cp4d_ref_adjoint)(self._ref(), _p(g), _p(f))
        return f

    def forward_rays(self, f, zkb):
        f = np.ascontiguousarray(f, dtype=np.float64)
        zkb = np.ascontiguousarray(zkb, dtype=np.int32).reshape(-1, 3)
        out = np.empty(len(zkb))
        lib().cp4d_ref_forward_rays(self._ref(), _p(f), C.c_int64(len(zkb)), zkb.ctypes.data_as(C.c_void_p), _p(out))
        return out

    def adjoint_voxels(self, g, zyx):
        g = np.ascontiguousarray(g, dtype=np.float64)
        zyx = np.ascontiguousarray(zyx, dtype=np.int32).reshape(-1, 3)
        out = np.empty((len(zyx), self.m))
        lib().cp4d_ref_adjoint_voxels(self._ref(), _p(g), C.c_int64(len(zyx)), zyx.ctypes.data_as(C.c_void_p), _p(out))
        return out

    def dense_A(self, k):
        """Static Joseph matrix of angle index k from the closed form, shape (nd, n*n)."""
        A = np.empty((self.nd, self.n * self.n))
        lib().cp4d_ref_dense_A(self._ref(), C.c_int(int(k)), _p(A))
        return A

    def grad(self, f):
        f = np.ascontiguousarray(f, dtype=np.float64)
        p = np.empty((4,) + self.primal_shape)
        lib().cp4d_ref_grad(self._ref(), _p(f), _p(p))
        return p

    def div(self, p):
        p = np.ascontiguousarray(p, dtype=np.float64)
        f = np.empty(self.primal_shape)
        lib().cp4d_ref_div(self._ref(), _p(p), _p(f))
        return f

    def prox_f1(self, h1, kf, g, sigma):
        h1 = np.array(h1, dtype=np.float64, order="C")
        lib().cp4d_ref_prox_f1(C.c_int64(h1.size), C.c_double(sigma), _p(np.ascontiguousarray(kf, dtype=np.float64)),
                               _p(np.ascontiguousarray(g, dtype=np.float64)), _p(h1))
        return h1

    def prox_f2(self, h2, gr, sigma, lambda1=None):
        h2 = np.array(h2, dtype=np.float64, order="C")
        lam = self.lambda1 if lambda1 is None else lambda1
        ncl = lib().cp4d_ref_prox_f2(C.c_int64(h2.size // 4), C.c_double(sigma), C.c_double(lam),
                                     _p(np.ascontiguousarray(gr, dtype=np.float64)), _p(h2))
        return h2, int(ncl)

    # iteration ------------------------------------------------------------------------------
    def zero_state(self):
        return dict(f=np.zeros(self.primal_shape), ft=np.zeros(self.primal_shape),
                    h1=np.zeros(self.sino_shape), h2=np.zeros((4,) + self.primal_shape))

    def cp(self, g, state, tau, sigma, n_iters, theta=1.0, folded=False):
        """Advance `state` (dict f, ft, h1, h2; modified in place) by n_iters iterations of Fig. 2."""
        g = np.ascontiguousarray(g, dtype=np.float64)
        ncl = lib().cp4d_ref_cp(self._ref(), _p(g), C.c_double(tau), C.c_double(sigma), C.c_double(theta),
                                C.c_int(int(n_iters)), C.c_int(int(folded)), _p(state["f"]), _p(state["ft"]),
                                _p(state["h1"]), _p(state["h2"]))
        return int(ncl)

    def power(self, x0, n_steps=30, use_k1=True, use_k2=True, folded=False):
        x = np.array(x0, dtype=np.float64, order="C")
        L = lib().cp4d_ref_power(self._ref(), _p(x), C.c_int(int(n_steps)), C.c_int(int(use_k1)),
                                 C.c_int(int(use_k2)), C.c_int(int(folded)))
        return float(L), x


class FrameProblem:
    """The paper's own temporal discretisation, TEST INFRASTRUCTURE like everything in oracle/.

    The primal variable is N_t time frames f(t_q) (4th axis of length N_t); frame q sits at the time of angle
    q*N_theta/N_t (Eq. 11).  The coefficients entering Eq. (9) are
        f_j = sum_q f(t_q) phi_j(t_q)                                              (L231-L237)
    i.e. f_coef = f_frames @ Psi^T with Psi[j,q] = phi_j(t_q) = Phi[j, q*N_theta/N_t], so
        K1' = K1 o analysis,   K1'^T = analysis^T o K1^T,
    and K2 differences the frames (L225-L227; the scale alpha/Delta_theta is absorbed in lambda2, R4).
    Written as plain numpy compositions of the operators of `Problem` (a matmul serves as the analysis step); the CP loop
    below is Fig. 2 (L147-L168) line by line.
    """

    def __init__(self, n, nz, nd, n_angles, n_half_rot, m, phi, n_frames, lambda1=1e-3, lambda2=1.0):
        assert n_angles % n_frames == 0
        self.coef = Problem(n, nz, nd, n_angles, n_half_rot, m, phi, lambda1, lambda2)
        self.psi = np.ascontiguousarray(np.asarray(phi, dtype=np.float64).reshape(m, n_angles)[:, ::n_angles // n_frames])
        # grad / div / proxes only see the array shape: a Problem whose 4th axis has n_frames entries
        self.frames = Problem(n, nz, nd, n_angles, n_half_rot, n_frames, np.zeros((n_frames, n_angles)), lambda1, lambda2)
        self.n_frames, self.lambda1, self.lambda2 = n_frames, lambda1, lambda2
        self.primal_shape, self.sino_shape = self.frames.primal_shape, self.coef.sino_shape

    def analysis(self, u):
        return np.ascontiguousarray(np.asarray(u, dtype=np.float64) @ self.psi.T)

    def analysis_t(self, f):
        return np.ascontiguousarray(np.asarray(f, dtype=np.float64) @ self.psi)

    def forward(self, u, folded=False):
        return self.coef.forward(self.analysis(u), folded=folded)

    def adjoint(self, g, folded=False):
        return self.analysis_t(self.coef.adjoint(g, folded=folded))

    def grad(self, u):
        return self.frames.grad(u)

    def div(self, p):
        return self.frames.div(p)

    def zero_state(self):
        return dict(f=np.zeros(self.primal_shape), ft=np.zeros(self.primal_shape),
                    h1=np.zeros(self.sino_shape), h2=np.zeros((4,) + self.primal_shape))

    def cp(self, g, state, tau, sigma, n_iters, theta=1.0, folded=False):
        """Fig. 2, steps 3-6, on the frames; returns the number of clamped 4-vectors of the last step 4."""
        g = np.asarray(g, dtype=np.float64)
        ncl = 0
        for _ in range(n_iters):
            state["h1"] = self.frames.prox_f1(state["h1"], self.forward(state["ft"], folded), g, sigma)          # step 3
            state["h2"], ncl = self.frames.prox_f2(state["h2"], self.grad(state["ft"]), sigma, self.lambda1)     # step 4
            f_new = state["f"] - tau * self.adjoint(state["h1"], folded) + tau * self.div(state["h2"])           # step 5
            state["ft"] = f_new + theta * (f_new - state["f"])                                                   # step 6
            state["f"] = f_new
        return ncl


def shepp_logan_kernel(nd):
    """h[n] = -2 / (pi^2 (4 n^2 - 1)), n = -(nd-1) .. nd-1: the Shepp-Logan filter sampled at unit bin spacing."""
    n = np.arange(-(nd - 1), nd, dtype=np.float64)
    return -2.0 / (np.pi ** 2 * (4.0 * n * n - 1.0))


def fbp_half_rotations(n, nz, nd, n_angles, n_half_rot, g):
    """Static filtered backprojection of every half-rotation, TEST INFRASTRUCTURE.

    out[z,iy,ix,q] = (pi/n0) sum_{i<n0} R*_{theta_i}(h_SL * g[z, q n0 + i, .]); R* is the Joseph backprojector of `Problem`
    (R3), reached through the box basis phi_q = 1 on half-rotation q, for which K1^T stacks the N_pi static
    backprojections.  Plain definition: direct convolution per row, then the pinned adjoint.
    """
    n0 = n_angles // n_half_rot
    g = np.asarray(g, dtype=np.float64)
    h = shepp_logan_kernel(nd)
    gf = np.empty_like(g)
    for z in range(nz):
        for k in range(n_angles):
            gf[z, k] = np.convolve(g[z, k], h)[nd - 1:2 * nd - 1]        # sum_b' h[b - b'] g[b']
    box = np.zeros((n_half_rot, n_angles))
    for q in range(n_half_rot):
        box[q, q * n0:(q + 1) * n0] = 1.0
    P = Problem(n, nz, nd, n_angles, n_half_rot, n_half_rot, box)
    return (np.pi / n0) * P.adjoint(gf)
