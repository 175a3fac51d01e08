"""Thin ctypes binding of libcp4d.so (include/cp4d.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; PyTorch is used for device memory
(`torch.empty(..., device="cuda")`), `data_ptr()` and the current stream.  There is no CPU fallback:
if the library is missing or the device is not sm_100, calls raise.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libcp4d.so"
_lib = None

OK, EINVAL, EWORKSPACE, EUNSUPPORTED, ECUDA, ESTATE, ENOMEM, EINTERNAL, ETOOLARGE = 0, -1, -2, -3, -4, -5, -6, -7, -8
STATIC_SCRATCH_BYTES = 32 << 20      # CP4D_STATIC_SCRATCH_BYTES of include/cp4d.h


class Cp4dError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"cp4d error {code}: {msg}")
        self.code = code


class Params(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("nd", C.c_int32),
                ("n_angles", C.c_int32), ("n_half_rot", C.c_int32), ("m", C.c_int32), ("device", C.c_int32),
                ("phi_host", C.c_void_p), ("lambda1", C.c_float), ("lambda2", C.c_float),
                ("theta_relax", C.c_float), ("workspace_dev", C.c_void_p), ("workspace_bytes", C.c_uint64),
                ("stream", C.c_void_p), ("n_frames", C.c_int32), ("z_open", C.c_int32)]


K_COUNT = 12


class Profile(C.Structure):
    _fields_ = [("ms", C.c_double * K_COUNT), ("launches", C.c_uint64 * K_COUNT)]


def lib():
    """Load libcp4d.so (built in-tree by paper_1809_09725_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise FileNotFoundError(f"{LIB_PATH} not built: run `python -c 'import __graft_entry__ as g; g.build()'` "
                                    "(no CPU fallback exists)")
        L = C.CDLL(str(LIB_PATH))
        vp, f32, i32, u64 = C.c_void_p, C.c_float, C.c_int32, C.c_uint64
        sig = {
            "cp4d_workspace_bytes": [C.POINTER(Params), C.POINTER(u64)],
            "cp4d_workspace_bytes_fused": [C.POINTER(Params), C.POINTER(u64)],
            "cp4d_fused_step_in_use": [vp, C.POINTER(i32)],
            "cp4d_create": [C.POINTER(Params), C.POINTER(vp)],
            "cp4d_destroy": [vp],
            "cp4d_forward": [vp, vp, vp], "cp4d_forward_static": [vp, vp, vp], "cp4d_adjoint": [vp, vp, vp], "cp4d_grad": [vp, vp, vp], "cp4d_div": [vp, vp, vp],
            "cp4d_prox_f1": [vp, f32, vp, vp, vp], "cp4d_prox_f2": [vp, f32, vp, vp],
            "cp4d_primal_update": [vp, f32, vp, vp, vp, vp],
            "cp4d_dot": [vp, vp, vp, u64, C.POINTER(C.c_double)],
            "cp4d_norm": [vp, i32, u64, C.POINTER(f32)],
            "cp4d_norm_start": [vp, i32, vp, C.POINTER(f32)],
            "cp4d_set_data": [vp, vp], "cp4d_set_steps": [vp, f32, f32], "cp4d_reset": [vp, vp],
            "cp4d_iterate": [vp, i32], "cp4d_get_f": [vp, vp],
            "cp4d_state_ptrs": [vp] + [C.POINTER(vp)] * 5,
            "cp4d_solve_host": [vp, vp, i32, vp], "cp4d_sync": [vp],
            "cp4d_objective": [vp] + [C.POINTER(C.c_double)] * 3, "cp4d_fbp": [vp, vp, vp],
            "cp4d_grad_slab": [vp, vp, vp, vp], "cp4d_div_slab": [vp, vp, vp, vp],
            "cp4d_step_dual": [vp, vp], "cp4d_step_primal": [vp, vp], "cp4d_set_z_open": [vp, i32],
            "cp4d_launch_count": [vp, C.POINTER(u64)],
            "cp4d_set_projector_mode": [vp, i32], "cp4d_projector_mode_in_use": [vp, C.POINTER(i32), C.POINTER(i32)],
            "cp4d_graph_replays": [vp, C.POINTER(u64)],
            "cp4d_profile_begin": [vp], "cp4d_profile_end": [vp, C.POINTER(Profile)],
        }
        for name, args in sig.items():
            fn = getattr(L, name)
            fn.argtypes, fn.restype = args, C.c_int
        for name in ("cp4d_strerror", "cp4d_last_error", "cp4d_version", "cp4d_kernel_name", "cp4d_graph_note"):
            getattr(L, name).restype = C.c_char_p
        L.cp4d_kernel_name.argtypes = [C.c_int]
        L.cp4d_strerror.argtypes = [C.c_int]
        L.cp4d_last_error.argtypes = [vp]
        L.cp4d_graph_note.argtypes = [vp]
        _lib = L
    return _lib


def make_params(n, nz, nd, n_angles, n_half_rot, m, phi=None, lambda1=1e-3, lambda2=1.0, theta=1.0, device=0,
                workspace_ptr=0, workspace_bytes=0, stream=0, ny=None, n_frames=0, z_open=0):
    p = Params()
    p.nx, p.ny, p.nz, p.nd = n, (n if ny is None else ny), nz, nd
    p.n_angles, p.n_half_rot, p.m, p.device = n_angles, n_half_rot, m, device
    p.phi_host = None if phi is None else phi.ctypes.data
    p.lambda1, p.lambda2, p.theta_relax = lambda1, lambda2, theta
    p.workspace_dev, p.workspace_bytes, p.stream = workspace_ptr or None, workspace_bytes, stream or None
    p.n_frames, p.z_open = n_frames, z_open
    return p


def workspace_bytes(n, nz, nd, n_angles, n_half_rot, m, n_frames=0, fused=False) -> int:
    """cp4d_workspace_bytes, or with fused=True cp4d_workspace_bytes_fused (second copies of h2 and ft for the one-pass step)."""
    out = C.c_uint64(0)
    p = make_params(n, nz, nd, n_angles, n_half_rot, m, n_frames=n_frames)
    r = (lib().cp4d_workspace_bytes_fused if fused else lib().cp4d_workspace_bytes)(C.byref(p), C.byref(out))
    if r:
        raise Cp4dError(r, lib().cp4d_strerror(r).decode())
    return out.value


class Context:
    """One reconstruction problem on one GPU.  Tensors are torch CUDA float32, contiguous, layouts of cp4d.h.
    fused=True allocates the workspace of cp4d_workspace_bytes_fused (5 V floats more), on which cp4d_iterate runs steps 4-6 of
    Fig. 2 as one kernel (13 V instead of 17 V floats of HBM traffic per iteration; same iterates); state() then returns the
    CURRENT copies of ft and h2, valid until the next iterate()."""

    def __init__(self, n, nz, nd, n_angles, n_half_rot, m, phi, lambda1=1e-3, lambda2=1.0, theta=1.0, device=0, n_frames=0,
                 z_open=0, fused=False):
        import torch
        self.torch = torch
        self.n, self.nz, self.nd, self.n_angles, self.n_half_rot, self.m = n, nz, nd, n_angles, n_half_rot, m
        self.n_frames, self.z_open = n_frames, z_open
        mp = n_frames or m                                   # length of the primal 4th axis (frames or coefficients)
        self.primal_shape, self.sino_shape = (nz, n, n, mp), (nz, n_angles, nd)
        self.V, self.S = nz * n * n * mp, nz * n_angles * nd
        self.device = torch.device("cuda", device)
        self._phi = np.ascontiguousarray(phi, dtype=np.float32).reshape(m, n_angles)
        # fused=True: a workspace with room for the one-pass step of cp4d_iterate (5 V floats more; whole-volume contexts only)
        nbytes = workspace_bytes(n, nz, nd, n_angles, n_half_rot, m, n_frames, fused=bool(fused) and not z_open)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self.workspace.data_ptr() + 255) // 256 * 256
            self.stream = torch.cuda.current_stream(self.device)
            p = make_params(n, nz, nd, n_angles, n_half_rot, m, self._phi, lambda1, lambda2, theta, device,
                            base, nbytes, self.stream.cuda_stream, n_frames=n_frames, z_open=z_open)
            h = C.c_void_p()
            r = lib().cp4d_create(C.byref(p), C.byref(h))
        if r:
            raise Cp4dError(r, lib().cp4d_strerror(r).decode())
        self._h = h

    @classmethod
    def from_config(cls, c, phi=None, device=0, n_frames=0, **kw):
        from . import synth
        if phi is None:
            phi = synth.basis_table(c.basis, c.m, c.n_angles)
        kw.setdefault("lambda1", c.lambda1)
        kw.setdefault("lambda2", c.lambda2)
        return cls(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m, phi, device=device, n_frames=n_frames, **kw)

    # -- helpers ---------------------------------------------------------------------------------
    def _ck(self, r):
        if r:
            raise Cp4dError(r, f"{lib().cp4d_strerror(r).decode()}: {lib().cp4d_last_error(self._h).decode()}")

    def _t(self, t, numel):
        assert t.is_cuda and t.dtype == self.torch.float32 and t.is_contiguous() and t.numel() == numel, \
            f"need contiguous cuda float32 tensor with {numel} elements, got {tuple(t.shape)} {t.dtype} {t.device}"
        return t.data_ptr()

    def empty_primal(self):
        return self.torch.empty(self.primal_shape, dtype=self.torch.float32, device=self.device)

    def empty_sino(self):
        return self.torch.empty(self.sino_shape, dtype=self.torch.float32, device=self.device)

    def empty_dual(self):
        return self.torch.empty((4,) + self.primal_shape, dtype=self.torch.float32, device=self.device)

    # -- operators (names of include/cp4d.h) -----------------------------------------------------
    def forward(self, f, out=None):
        out = self.empty_sino() if out is None else out
        self._ck(lib().cp4d_forward(self._h, self._t(f, self.V), self._t(out, self.S)))
        return out

    def forward_static(self, f, out=None):
        """cp4d_forward with the projector's scratch in the library's static device array (no workspace scratch at call time)."""
        out = self.empty_sino() if out is None else out
        self._ck(lib().cp4d_forward_static(self._h, self._t(f, self.V), self._t(out, self.S)))
        return out

    def adjoint(self, g, out=None):
        out = self.empty_primal() if out is None else out
        self._ck(lib().cp4d_adjoint(self._h, self._t(g, self.S), self._t(out, self.V)))
        return out

    def grad(self, f, out=None):
        out = self.empty_dual() if out is None else out
        self._ck(lib().cp4d_grad(self._h, self._t(f, self.V), self._t(out, 4 * self.V)))
        return out

    def div(self, p, out=None):
        out = self.empty_primal() if out is None else out
        self._ck(lib().cp4d_div(self._h, self._t(p, 4 * self.V), self._t(out, self.V)))
        return out

    # -- z-slab contexts (z_open != 0): the neighbour's slice enters as a one-slice tensor or a raw device pointer ----
    def _halo(self, h):
        if h is None or isinstance(h, int):
            return h or None
        return self._t(h, self.V // self.nz)

    def set_z_open(self, z_open):
        self._ck(lib().cp4d_set_z_open(self._h, z_open))
        self.z_open = z_open

    def grad_slab(self, f, f_above=None, out=None):
        out = self.empty_dual() if out is None else out
        self._ck(lib().cp4d_grad_slab(self._h, self._t(f, self.V), self._halo(f_above), self._t(out, 4 * self.V)))
        return out

    def div_slab(self, p, pz_below=None, out=None):
        out = self.empty_primal() if out is None else out
        self._ck(lib().cp4d_div_slab(self._h, self._t(p, 4 * self.V), self._halo(pz_below), self._t(out, self.V)))
        return out

    def step_dual(self, ft_above=None):
        self._ck(lib().cp4d_step_dual(self._h, self._halo(ft_above)))

    def step_primal(self, h2z_below=None):
        self._ck(lib().cp4d_step_primal(self._h, self._halo(h2z_below)))

    def prox_f1(self, sigma, ft, g, h1):
        self._ck(lib().cp4d_prox_f1(self._h, sigma, self._t(ft, self.V), self._t(g, self.S), self._t(h1, self.S)))
        return h1

    def prox_f2(self, sigma, ft, h2):
        self._ck(lib().cp4d_prox_f2(self._h, sigma, self._t(ft, self.V), self._t(h2, 4 * self.V)))
        return h2

    def primal_update(self, tau, h1, h2, f, ft):
        self._ck(lib().cp4d_primal_update(self._h, tau, self._t(h1, self.S), self._t(h2, 4 * self.V),
                                          self._t(f, self.V), self._t(ft, self.V)))
        return f, ft

    def dot(self, x, y):
        out = C.c_double(0)
        assert x.numel() == y.numel()
        self._ck(lib().cp4d_dot(self._h, self._t(x, x.numel()), self._t(y, y.numel()), x.numel(), C.byref(out)))
        return out.value

    def norm(self, n_power_iters=30, seed=0):
        out = C.c_float(0)
        self._ck(lib().cp4d_norm(self._h, n_power_iters, seed, C.byref(out)))
        return out.value

    def norm_start(self, x0, n_power_iters=30):
        """Power iteration from the caller's start vector x0 (primal-shaped cuda tensor; copied, not modified)."""
        out = C.c_float(0)
        self._ck(lib().cp4d_norm_start(self._h, n_power_iters, self._t(x0, self.V), C.byref(out)))
        return out.value

    # -- CP state machine ------------------------------------------------------------------------
    def set_data(self, g):
        self._ck(lib().cp4d_set_data(self._h, self._t(g, self.S)))

    def set_steps(self, tau, sigma):
        self._ck(lib().cp4d_set_steps(self._h, tau, sigma))

    def reset(self, f0=None):
        self._ck(lib().cp4d_reset(self._h, None if f0 is None else self._t(f0, self.V)))

    def iterate(self, n_iters):
        self._ck(lib().cp4d_iterate(self._h, n_iters))

    def get_f(self, out=None):
        out = self.empty_primal() if out is None else out
        self._ck(lib().cp4d_get_f(self._h, self._t(out, self.V)))
        return out

    def state(self):
        """Views (no copy) of the state arrays inside the workspace: dict f, ft, h1, h2, g."""
        ptrs = [C.c_void_p() for _ in range(5)]
        self._ck(lib().cp4d_state_ptrs(self._h, *[C.byref(p) for p in ptrs]))
        base = self.workspace.data_ptr()
        shapes = [self.primal_shape, self.primal_shape, self.sino_shape, (4,) + self.primal_shape, self.sino_shape]
        out = {}
        for name, p, shp in zip(("f", "ft", "h1", "h2", "g"), ptrs, shapes):
            off = p.value - base
            nb = int(np.prod(shp)) * 4
            out[name] = self.workspace[off:off + nb].view(self.torch.float32).view(shp)
        return out

    def solve_host(self, g_host, n_iters, f_host):
        """g_host / f_host: CPU float32 torch tensors (pinned for full copy speed) or numpy arrays."""
        gp = g_host.data_ptr() if hasattr(g_host, "data_ptr") else g_host.ctypes.data
        fp = f_host.data_ptr() if hasattr(f_host, "data_ptr") else f_host.ctypes.data
        self._ck(lib().cp4d_solve_host(self._h, gp, n_iters, fp))
        return f_host

    def fbp(self, g, out=None):
        """Static Shepp-Logan FBP of every half-rotation: (nz, n, n, 4*ceil(n_half_rot/4))."""
        q4 = (self.n_half_rot + 3) // 4 * 4
        if out is None:
            out = self.torch.empty((self.nz, self.n, self.n, q4), dtype=self.torch.float32, device=self.device)
        self._ck(lib().cp4d_fbp(self._h, self._t(g, self.S), self._t(out, self.nz * self.n * self.n * q4)))
        return out

    def objective(self):
        """(primal value, conditional dual value, dual residual |K1^T h1 - div h2|) of the current state; syncs."""
        out = [C.c_double(0) for _ in range(3)]
        self._ck(lib().cp4d_objective(self._h, *[C.byref(o) for o in out]))
        return tuple(o.value for o in out)

    def sync(self):
        self._ck(lib().cp4d_sync(self._h))

    def launch_count(self) -> int:
        out = C.c_uint64(0)
        self._ck(lib().cp4d_launch_count(self._h, C.byref(out)))
        return out.value

    def fused_step_in_use(self) -> bool:
        out = C.c_int32(0)
        self._ck(lib().cp4d_fused_step_in_use(self._h, C.byref(out)))
        return bool(out.value)

    def graph_replays(self) -> int:
        """CUDA-graph replays of one CP iteration issued by iterate() so far (0 on the legacy default stream)."""
        out = C.c_uint64(0)
        self._ck(lib().cp4d_graph_replays(self._h, C.byref(out)))
        return out.value

    def set_projector_mode(self, mode):
        """"auto" (tensor-core forward projector where it applies: m = 4, 8, 16, 32; fp32 backprojector), "fp32" (CUDA-core
        kernels on both sides) or "tensor" (tensor-core kernels on both sides where they apply)."""
        self._ck(lib().cp4d_set_projector_mode(self._h, {"auto": 0, "fp32": 1, "tensor": 2}[mode]))

    def projector_mode_in_use(self):
        """(forward, adjoint), each "fp32" or "tensor"."""
        fw, ad = C.c_int32(0), C.c_int32(0)
        self._ck(lib().cp4d_projector_mode_in_use(self._h, C.byref(fw), C.byref(ad)))
        return {1: "fp32", 2: "tensor"}[fw.value], {1: "fp32", 2: "tensor"}[ad.value]

    def graph_note(self) -> str:
        """Why iterate() is not replaying a CUDA graph ("" if it is, or has not tried yet)."""
        return lib().cp4d_graph_note(self._h).decode()

    def profile_begin(self):
        self._ck(lib().cp4d_profile_begin(self._h))

    def profile_end(self) -> dict:
        """{kernel class name: (summed device ms, timed launches)} since profile_begin; syncs."""
        pr = Profile()
        self._ck(lib().cp4d_profile_end(self._h, C.byref(pr)))
        return {lib().cp4d_kernel_name(k).decode(): (pr.ms[k], int(pr.launches[k])) for k in range(K_COUNT) if pr.launches[k]}

    def close(self):
        if getattr(self, "_h", None):
            lib().cp4d_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
