"""C-ABI boundary checks that need no GPU: the library loads, exports every symbol include/cp4d.h declares,
validates arguments on the host, and refuses to create a context without an sm_100 device (no CPU fallback)."""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parents[1]


@pytest.fixture(scope="module")
def L():
    from paper_1809_09725_b200 import build, binding
    build.build_lib()
    return binding.lib()


def declared_symbols():
    hdr = (ROOT / "include" / "cp4d.h").read_text()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    return sorted(set(re.findall(r"\b(cp4d_[a-z0-9_]+)\s*\(", hdr)))


def test_exports_every_declared_symbol(L):
    syms = declared_symbols()
    assert {"cp4d_create", "cp4d_forward", "cp4d_adjoint", "cp4d_grad", "cp4d_div", "cp4d_iterate", "cp4d_norm"} <= set(syms)
    for s in syms:
        assert hasattr(L, s), f"libcp4d.so does not export {s}"


def test_workspace_bytes_counts_state(L):
    from paper_1809_09725_b200 import binding, synth
    for cfg in (1, 2, 3, 4, 5):
        c = synth.CONFIGS[cfg]
        nb = binding.workspace_bytes(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m)
        state = (7 * c.V + 3 * c.S) * 4                       # f, ft, K1^T h1, h2[4], h1, g, sinogram temporary
        # projector scratch rows are padded so that every tile window is readable memory (include/cp4d.h):
        # at most (sqrt2 (n-1) - (nd-1))/2 + 3 bins each side plus one window of 56 bins
        pad = 2 * (int(np.ceil(max(0.0, 0.5 * (np.sqrt(2.0) * (c.n - 1) - (c.nd - 1))))) + 3) + 56
        pitch = c.nd + pad + (1 if (c.nd + pad) % 8 == 0 else 0)
        scratch = c.nz * c.n_theta0 * pitch * c.m * 4          # folded sinogram of the adjoint (zero-padded rows)
        if c.m in (4, 8, 16, 32):
            # the tensor backprojector keeps it as split bf16 pairs, bin-major with one 16-byte unit of padding per bin:
            # 4 nb + 1 units per bin for groups of nb 16-entry batch blocks (whole z-groups)
            blocks = (c.nz * c.m + 15) // 16
            nblk = 4 if blocks >= 4 else 2 if blocks >= 2 else 1
            zper = nblk * 16 // c.m
            scratch = max(scratch, -(-c.nz // zper) * c.n_theta0 * (4 * nblk + 1) * pitch * 16)
        scratch += c.nz * c.n_theta0 * c.nd * c.m * 4          # partial ray sums of the forward projector (no padding)
        # work items of the tensor forward projector, built once per context: per 32 x 32 tile, 4 x 14 items of 48 bytes
        # for each of at most n_theta0 / 4 + 8 angle groups (groups of four from 72 base angles on, pairs from 24)
        gs = 4 if c.n_theta0 >= 72 else 2 if c.n_theta0 >= 24 else 1
        tiles = ((c.n + 31) // 32) ** 2
        scratch += tiles * 4 * 14 * (c.n_theta0 // gs + 8) * 48
        scratch += tiles * 2 * (c.n_theta0 + 8) * 32           # angle records of the tensor backprojector per (half tile, angle)
        assert state + scratch <= nb <= state + scratch + (64 << 20)
        # the one-pass step of cp4d_iterate double-buffers h2[4] and ft: 5 V floats more
        nbf = binding.workspace_bytes(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m, fused=True)
        assert 5 * c.V * 4 <= nbf - nb <= 5 * c.V * 4 + 512
    c = synth.CONFIGS[5]
    assert binding.workspace_bytes(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m, fused=True) < 170e9   # fits 180 GB HBM


@pytest.mark.parametrize("bad", [dict(ny=31), dict(m=6), dict(m=36), dict(n_half_rot=3), dict(nd=1), dict(nz=0), dict(lambda1=-1.0),
                                 dict(n_frames=6), dict(n_frames=-4), dict(n_frames=12), dict(n_frames=36)])
def test_host_validation(L, bad):
    from paper_1809_09725_b200 import binding
    kw = dict(n=32, nz=1, nd=32, n_angles=128, n_half_rot=4, m=4)
    kw.update(bad)
    p = binding.make_params(**kw)
    out = C.c_uint64(0)
    assert L.cp4d_workspace_bytes(C.byref(p), C.byref(out)) == binding.EINVAL


def test_phi_slice_must_fit_shared_memory(L):
    """k_fold / k_synth stage the n_half_rot x m slice of Phi in 48 KB of shared memory: larger products are refused at
    validation instead of failing at the first launch."""
    from paper_1809_09725_b200 import binding
    out = C.c_uint64(0)
    ok = binding.make_params(n=32, nz=1, nd=32, n_angles=384 * 2, n_half_rot=384, m=32)
    assert L.cp4d_workspace_bytes(C.byref(ok), C.byref(out)) == binding.OK
    bad = binding.make_params(n=32, nz=1, nd=32, n_angles=385 * 2, n_half_rot=385, m=32)
    assert L.cp4d_workspace_bytes(C.byref(bad), C.byref(out)) == binding.EINVAL


def test_frame_mode_workspace(L):
    """Frame mode (n_frames > 0).  N_t <= M collapses to a coefficient-mode problem with N_t planes (the projector pair carries
    the frames); N_t > M keeps M-plane coefficient stacks beside the N_t-plane state plus the Psi table."""
    from paper_1809_09725_b200 import binding
    n, nz, nd, na, npi = 64, 4, 64, 96, 2
    assert binding.workspace_bytes(n, nz, nd, na, npi, 16, n_frames=8) == binding.workspace_bytes(n, nz, nd, na, npi, 8)
    a = binding.workspace_bytes(n, nz, nd, na, npi, 4)
    b = binding.workspace_bytes(n, nz, nd, na, npi, 4, n_frames=8)
    vox = nz * n * n
    assert b - a == pytest.approx((7 * (8 - 4) + 2 * 4) * vox * 4, abs=1 << 16)


def test_create_needs_workspace_and_device(L):
    from paper_1809_09725_b200 import binding
    import torch
    phi = np.ones((4, 128), dtype=np.float32)
    p = binding.make_params(32, 1, 32, 128, 4, 4, phi)
    h = C.c_void_p()
    assert L.cp4d_create(C.byref(p), C.byref(h)) == binding.EWORKSPACE
    if not torch.cuda.is_available():
        p = binding.make_params(32, 1, 32, 128, 4, 4, phi, workspace_ptr=4096, workspace_bytes=1 << 30)
        assert L.cp4d_create(C.byref(p), C.byref(h)) == binding.EUNSUPPORTED      # fails loudly: no CPU fallback
        assert h.value is None
    assert L.cp4d_forward(None, None, None) == binding.EINVAL
    assert L.cp4d_strerror(binding.EUNSUPPORTED).decode().startswith("no sm_100")


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (it is test infrastructure)."""
    for p in list((ROOT / "paper_1809_09725_b200").rglob("*.py")) + list((ROOT / "paper_1809_09725_b200" / "csrc").glob("*.cu*")):
        txt = p.read_text()
        assert not re.search(r"^\s*(from|import)\s+oracle|libcp4d_ref|cp4d_ref_|oracle[./]ref", txt, flags=re.M), \
            f"{p} reaches into the oracle"
