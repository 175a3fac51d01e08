"""Host logic of the z-slab decomposition (paper_1809_09725_b200/slabs.py) on the CPU.

The halo protocol (which slice is sent when) is run with world_size 2 over gloo: each rank owns one slab whose step calls
are built from the ORACLE's operators on an extended array (a neighbour slice appended / prepended), the slices travel
through slabs.exchange_halos, and the result must equal the oracle's whole-volume Chambolle-Pock run."""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parents[1]


def test_partition_covers_every_slice_once():
    from paper_1809_09725_b200 import slabs
    for nz in (1, 2, 5, 32, 33):
        for k in range(1, min(nz, 7) + 1):
            r = slabs.partition(nz, k)
            assert r[0][0] == 0 and r[-1][1] == nz and all(a[1] == b[0] for a, b in zip(r, r[1:]))
            sizes = [b - a for a, b in r]
            assert min(sizes) >= 1 and max(sizes) - min(sizes) <= 1
            flags = [slabs.z_open_flags(i, k) for i in range(k)]
            assert flags[0] & 1 == 0 and flags[-1] & 2 == 0 and all(f == 3 for f in flags[1:-1])
    with pytest.raises(ValueError):
        slabs.partition(3, 4)


class OracleSlab:
    """A slab whose steps are the oracle's operators; the neighbour slices enter by extending the arrays along z."""

    def __init__(self, P, g, tau, sigma, lo_open, hi_open):
        import torch
        self.P, self.g, self.tau, self.sigma, self.lo, self.hi = P, g, tau, sigma, lo_open, hi_open
        self.st = P.zero_state()
        one = (1,) + P.primal_shape[1:]
        self.ft_above = torch.zeros(P.primal_shape[1:], dtype=torch.float64)
        self.h2z_below = torch.zeros(P.primal_shape[1:], dtype=torch.float64)
        self._one = one
        self._ext = {}

    def _problem(self, nz):
        if nz not in self._ext:
            P = self.P
            self._ext[nz] = type(P)(P.n, nz, P.nd, P.n_angles, P.n_half_rot, P.m, P.phi, lambda1=P.lambda1, lambda2=P.lambda2)
        return self._ext[nz]

    def ft_first(self):
        import torch
        return torch.from_numpy(np.ascontiguousarray(self.st["ft"][0]))

    def h2z_last(self):
        import torch
        return torch.from_numpy(np.ascontiguousarray(self.st["h2"][2, -1]))

    def step_dual(self, halo):
        P, st = self.P, self.st
        assert (halo is not None) == self.hi
        st["h1"] = P.prox_f1(st["h1"], P.forward(st["ft"], folded=True), self.g, self.sigma)
        if halo is None:
            gr = P.grad(st["ft"])
        else:      # one more slice on top: the z-difference of the slab's last slice sees the neighbour
            ext = np.concatenate([st["ft"], halo.numpy().reshape(self._one)], axis=0)
            gr = self._problem(ext.shape[0]).grad(ext)[:, :-1]
        st["h2"], _ = P.prox_f2(st["h2"], gr, self.sigma)

    def step_primal(self, halo):
        P, st = self.P, self.st
        assert (halo is not None) == self.lo
        p = st["h2"]
        lead = np.zeros((4,) + self._one)
        if halo is not None:
            lead[2, 0] = halo.numpy()
        # a zero slice on top makes the slab's last p_z interior (hi_open); a leading slice carries the neighbour's p_z
        parts = ([lead] if self.lo else []) + [p] + ([np.zeros((4,) + self._one)] if self.hi else [])
        ext = np.concatenate(parts, axis=1)
        d = self._problem(ext.shape[1]).div(ext)[(1 if self.lo else 0):(ext.shape[1] - (1 if self.hi else 0))]
        fn = st["f"] - self.tau * P.adjoint(st["h1"], folded=True) + self.tau * d
        st["ft"] = fn + 1.0 * (fn - st["f"])
        st["f"] = fn


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, str(ROOT))
    from oracle import ref
    from paper_1809_09725_b200 import slabs, synth
    ref.build(); ref.set_threads(1)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    c = synth.CONFIGS[1].scaled(cfg=31, n=12, nd=14, nz=5, n_angles=12, n_half_rot=2, m=4, lambda1=0.02, lambda2=0.8)
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    g = synth.rng(c.cfg, 2).standard_normal((c.nz, c.n_angles, c.nd))
    z0, z1 = slabs.partition(c.nz, world)[rank]
    P = ref.Problem.from_config(c.scaled(nz=z1 - z0), phi=phi)
    flags = slabs.z_open_flags(rank, world)
    slab = OracleSlab(P, g[z0:z1], 0.03, 0.04, bool(flags & 1), bool(flags & 2))
    slabs.iterate_rank(slab, rank, world, 6)
    dist.barrier()
    out.put((rank, z0, z1, slab.st["f"], slab.st["h2"]))
    dist.destroy_process_group()


def test_halo_protocol_gloo_world2_matches_whole_volume_oracle(oracle):
    import torch.multiprocessing as mp
    from paper_1809_09725_b200 import synth
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=240) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    c = synth.CONFIGS[1].scaled(cfg=31, n=12, nd=14, nz=5, n_angles=12, n_half_rot=2, m=4, lambda1=0.02, lambda2=0.8)
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    g = synth.rng(c.cfg, 2).standard_normal((c.nz, c.n_angles, c.nd))
    P = oracle.Problem.from_config(c, phi=phi)
    st = P.zero_state()
    ncl = P.cp(g, st, 0.03, 0.04, 6, folded=True)
    assert 0 < ncl < P.V                               # both branches of the F2* prox are active
    f = np.concatenate([r[3] for r in res], axis=0)
    h2 = np.concatenate([r[4] for r in res], axis=1)
    assert np.abs(f - st["f"]).max() <= 1e-12 * np.abs(st["f"]).max()
    assert np.abs(h2 - st["h2"]).max() <= 1e-12 * np.abs(st["h2"]).max()
    # and the z-coupling is really exercised: without the halos the slabs give a different answer
    assert np.abs(st["h2"][2, res[0][2] - 1]).max() > 0


def test_temporal_blocking_windows_keep_the_core_exact(oracle):
    """The claim slabs.StreamedSolver.windows rests on: k iterations of a CLOSED window of slices spoil exactly k slices next to
    each interior window end, so a core at distance >= k is the whole-volume iterate.  Checked with the oracle: every slab's window
    iterated on its own equals the whole-volume run on its core, and the slice just outside the safe distance does not."""
    from paper_1809_09725_b200 import slabs, synth
    c = synth.CONFIGS[1].scaled(cfg=32, n=10, nd=12, nz=11, n_angles=8, n_half_rot=2, m=4, lambda1=0.02, lambda2=0.8)
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    g = synth.rng(c.cfg, 2).standard_normal((c.nz, c.n_angles, c.nd))
    k = 3
    P = oracle.Problem.from_config(c, phi=phi)
    whole = P.zero_state()
    P.cp(g, whole, 0.03, 0.04, 2, folded=True)          # a non-trivial starting iterate n
    start = {a: v.copy() for a, v in whole.items()}
    assert 0 < P.cp(g, whole, 0.03, 0.04, k, folded=True) < P.V

    class Geo:                                          # the window arithmetic of StreamedSolver without a device
        block, nz, slab_nz = k, c.nz, 2
    Geo.win_nz = min(c.nz, Geo.slab_nz + 2 * k)
    Geo.ranges = [(i * 2, min(c.nz, i * 2 + 2)) for i in range((c.nz + 1) // 2)]
    wins = slabs.StreamedSolver.windows(Geo)
    assert [w[2:] for w in wins] == Geo.ranges and all(w1 - w0 == Geo.win_nz for w0, w1, _, _ in wins)
    spoiled = 0
    for w0, w1, z0, z1 in wins:
        assert (w0 == 0 or z0 - w0 >= k) and (w1 == c.nz or w1 - z1 >= k)
        Pw = oracle.Problem.from_config(c.scaled(nz=w1 - w0), phi=phi)
        st = {a: np.array(v[:, w0:w1] if a == "h2" else v[w0:w1], order="C") for a, v in start.items()}   # copies: cp works in place
        Pw.cp(g[w0:w1], st, 0.03, 0.04, k, folded=True)
        for a in ("f", "ft", "h1"):
            assert np.array_equal(st[a][z0 - w0:z1 - w0], whole[a][z0:z1]), a
        assert np.array_equal(st["h2"][:, z0 - w0:z1 - w0], whole["h2"][:, z0:z1])
        if w0 > 0:                                      # one slice closer than k to the interior end is already wrong
            spoiled += not np.array_equal(st["f"][k - 1], whole["f"][w0 + k - 1])
    assert spoiled > 0
