"""z-slab decomposition of the Chambolle-Pock iteration.

K1, K1^T and the x/y/t differences act per slice; only the z-difference of K2 / K2^T couples neighbouring slices.  The
volume is cut into contiguous z-slabs, one cp4d context (`cp4d_params.z_open`) per slab, and per iteration a slab needs two
read-only slices from its neighbours (L283: "two extra slices located before and after the current set of slices"):

    dual step   (Fig. 2 steps 3-4): the upper neighbour's first slice of ft, as it was before this iteration's update
    primal step (Fig. 2 steps 5-6): the lower neighbour's last slice of the z-component of h2, after this iteration's prox

Three drivers of the same two calls (`cp4d_step_dual`, `cp4d_step_primal`); argument marshalling and copies only, every step
of the path runs in the library's kernels:

  SlabSolver      all slabs resident on one GPU; a halo is the neighbour's state slice itself (no copy), so the slabs
                  run in two phases: every dual step, then every primal step.
  StreamedSolver  the state lives in pinned HOST memory and passes through a small pool of device slabs, for volumes beyond HBM
                  (L285: one stream each for host-to-device copies, compute, device-to-host copies).  One sweep in increasing z
                  per iteration: slab s runs dual + primal back to back; its ft halo is the OLD first slice of slab s+1 (not yet
                  updated on the host), its h2z halo the NEW last slice of slab s-1 (kept on the device from the previous slab).
  exchange_halos  one slab per rank (`torch.distributed`): the two halo slices as send/recv pairs between z-neighbours.
"""
from __future__ import annotations

import numpy as np

from . import binding


def partition(nz: int, n_slabs: int):
    """Contiguous z-ranges [(z0, z1), ...] of nearly equal size (L283: slab i = slices i*Nz/Nth ... (i+1)*Nz/Nth - 1)."""
    if not (1 <= n_slabs <= nz):
        raise ValueError(f"need 1 <= n_slabs <= nz, got {n_slabs} slabs for {nz} slices")
    cuts = [(i * nz) // n_slabs for i in range(n_slabs + 1)]
    return [(cuts[i], cuts[i + 1]) for i in range(n_slabs)]


def z_open_flags(i: int, n_slabs: int) -> int:
    """cp4d_params.z_open of slab i: bit 0 = lower face interior, bit 1 = upper face interior."""
    return (1 if i > 0 else 0) | (2 if i < n_slabs - 1 else 0)


class SlabSolver:
    """All slabs on one device.  Same results as one whole-volume Context (tests/test_gpu_slabs.py)."""

    def __init__(self, n, nz, nd, n_angles, n_half_rot, m, phi, n_slabs=2, device=0, **kw):
        self.ranges = partition(nz, n_slabs)
        self.nz, self.n_slabs = nz, n_slabs
        self.ctx = [binding.Context(n, z1 - z0, nd, n_angles, n_half_rot, m, phi, device=device,
                                    z_open=z_open_flags(i, n_slabs), **kw)
                    for i, (z0, z1) in enumerate(self.ranges)]
        self.torch = self.ctx[0].torch
        self._st = [c.state() for c in self.ctx]

    @classmethod
    def from_config(cls, c, phi=None, n_slabs=2, device=0, n_frames=0, **kw):
        from . import synth
        if phi is None:
            phi = synth.basis_table(c.basis, c.m, c.n_angles)
        kw.setdefault("lambda1", c.lambda1)
        kw.setdefault("lambda2", c.lambda2)
        return cls(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m, phi, n_slabs=n_slabs, device=device, n_frames=n_frames, **kw)

    def close(self):
        for c in self.ctx:
            c.close()

    # halos: views into the neighbours' state (same device, same stream: ordering is the stream's)
    def _ft_above(self, i):
        return self._st[i + 1]["ft"][0] if i + 1 < self.n_slabs else None

    def _h2z_below(self, i):
        return self._st[i - 1]["h2"][2, -1] if i > 0 else None

    def split(self, t):
        """Per-slab contiguous pieces of a tensor whose first axis is z: primal [z][y][x][j] and sinogram [z][k][b] tensors; dual
        tensors [4][z][y][x][j] (5 axes) are cut along axis 1.  Chosen by the number of axes, never by comparing sizes (nz = 4
        would be ambiguous)."""
        if t.dim() == 5:
            return [t[:, z0:z1].contiguous() for z0, z1 in self.ranges]
        return [t[z0:z1].contiguous() for z0, z1 in self.ranges]

    def set_data(self, g):
        for c, gs in zip(self.ctx, self.split(g)):
            c.set_data(gs)

    def set_steps(self, tau, sigma):
        for c in self.ctx:
            c.set_steps(tau, sigma)

    def reset(self, f0=None):
        parts = self.split(f0) if f0 is not None else [None] * self.n_slabs
        for c, p in zip(self.ctx, parts):
            c.reset(p)

    def iterate(self, n_iters):
        for _ in range(n_iters):
            for i, c in enumerate(self.ctx):           # phase 1: every ft halo is still the old iterate
                c.step_dual(self._ft_above(i))
            for i, c in enumerate(self.ctx):           # phase 2: every h2 is the new one
                c.step_primal(self._h2z_below(i))

    def gather(self, name):
        return self.torch.cat([s[name] for s in self._st], dim=1 if name == "h2" else 0)

    def get_f(self):
        return self.gather("f")

    def sync(self):
        for c in self.ctx:
            c.sync()

    def launch_count(self):
        return sum(c.launch_count() for c in self.ctx)

    # ---- operators on sharded tensors (lists of per-slab tensors) -------------------------------
    def grad(self, fs):
        return [c.grad_slab(f, fs[i + 1][0] if i + 1 < self.n_slabs else None) for i, (c, f) in enumerate(zip(self.ctx, fs))]

    def div(self, ps):
        return [c.div_slab(p, ps[i - 1][2, -1] if i > 0 else None) for i, (c, p) in enumerate(zip(self.ctx, ps))]

    def norm(self, n_power_iters=30, seed=0):
        """||K|| of the WHOLE volume by the power iteration of cp4d_norm (R8) on the sharded operators; the
        squared norms of the slabs are added on the host."""
        torch = self.torch
        gen = torch.Generator(device=self.ctx[0].device)
        gen.manual_seed(seed)
        xs = [torch.randn(c.primal_shape, generator=gen, device=c.device, dtype=torch.float32) for c in self.ctx]
        nrm = np.sqrt(sum(c.dot(x, x) for c, x in zip(self.ctx, xs)))
        xs = [x / nrm for x in xs]
        L = 0.0
        for _ in range(n_power_iters):
            y1 = [c.adjoint(c.forward(x)) for c, x in zip(self.ctx, xs)]          # K1^T K1 x
            y2 = self.div(self.grad(xs))                                          # -K2^T K2 x
            ys = [a - b for a, b in zip(y1, y2)]
            ny = np.sqrt(sum(c.dot(y, y) for c, y in zip(self.ctx, ys)))
            L = np.sqrt(ny)
            if not ny > 0.0:
                break
            xs = [y / ny for y in ys]
        return float(L)


class StreamedSolver:
    """CP iterations with the state in pinned host memory, streamed slab by slab through the GPU (volumes beyond HBM).

    Host arrays (torch CPU tensors, pinned): f, ft (nz, n, n, mp), h2 (4, nz, n, n, mp), h1, g (nz, n_angles, nd).
    Device: `depth` slab contexts (default 2) used round-robin; copies in on `s_in`, kernels on each context's stream,
    copies out on `s_out`, ordered by events, so the upload of slab s+1 and the download of slab s-1 overlap the kernels of
    slab s.  All slabs but the last have the same height, so at most two distinct context shapes are needed per pool slot.

    block = k > 1 (temporal blocking): a window of slab_nz + 2k slices is uploaded, iterated k times as a closed volume and
    only its core of slab_nz slices is written back (to a second host copy, since the neighbours still need iterate n): k times
    less PCIe traffic per iteration for (slab_nz + 2k) / slab_nz more kernel work.  See `windows`.
    """

    def __init__(self, n, nz, nd, n_angles, n_half_rot, m, phi, slab_nz, device=0, depth=2, n_frames=0, block=1, **kw):
        import torch
        self.torch = torch
        self.dev = torch.device("cuda", device)
        self.block, self.slab_nz = max(1, int(block)), slab_nz
        self.win_nz = min(nz, slab_nz + 2 * self.block)      # temporal blocking: slices per device window
        self.n, self.nz, self.nd, self.na = n, nz, nd, n_angles
        self.mp = n_frames or m
        n_slabs = (nz + slab_nz - 1) // slab_nz
        self.ranges = [(i * slab_nz, min(nz, (i + 1) * slab_nz)) for i in range(n_slabs)]
        self.n_slabs, self.depth = n_slabs, max(1, min(depth, n_slabs))
        self._mk = lambda h, stream: self._make_ctx(n, h, nd, n_angles, n_half_rot, m, phi, device, n_frames, stream, kw)
        self.s_in, self.s_out = torch.cuda.Stream(self.dev), torch.cuda.Stream(self.dev)
        self.s_cmp = [torch.cuda.Stream(self.dev) for _ in range(self.depth)]
        self._ctx = {}                                   # (slot, height) -> Context; the interior faces are set per slab
        pin = lambda *shape: torch.zeros(shape, dtype=torch.float32).pin_memory()
        self.f, self.ft = pin(nz, n, n, self.mp), pin(nz, n, n, self.mp)
        self.h2 = pin(4, nz, n, n, self.mp)
        self.h1, self.g = pin(nz, n_angles, nd), pin(nz, n_angles, nd)
        # temporal blocking reads iterate n and writes iterate n + block: a second host copy of the state
        self._nxt = dict(f=pin(nz, n, n, self.mp), ft=pin(nz, n, n, self.mp), h2=pin(4, nz, n, n, self.mp),
                         h1=pin(nz, n_angles, nd)) if self.block > 1 else None
        dev_buf = lambda *shape: torch.empty(shape, dtype=torch.float32, device=self.dev)
        self.halo_ft = [dev_buf(n, n, self.mp) for _ in range(self.depth)]
        self.halo_h2z = [dev_buf(n, n, self.mp) for _ in range(2)]
        self.g_stage = [dev_buf(self.win_nz if self.block > 1 else slab_nz, n_angles, nd) for _ in range(self.depth)]
        self.tau = self.sigma = None
        self.bytes_h2d = self.bytes_d2h = 0

    def _make_ctx(self, n, h, nd, na, npi, m, phi, device, n_frames, stream, kw):
        with self.torch.cuda.stream(stream):
            return binding.Context(n, h, nd, na, npi, m, phi, device=device, n_frames=n_frames, z_open=0, **kw)

    def _context(self, slot, i):
        z0, z1 = self.ranges[i]
        key = (slot, z1 - z0)                            # every slab but possibly the last has the same height
        if key not in self._ctx:
            c = self._mk(z1 - z0, self.s_cmp[slot])
            if self.tau is not None:
                c.set_steps(self.tau, self.sigma)
            self._ctx[key] = c
        c = self._ctx[key]
        c.set_z_open(z_open_flags(i, self.n_slabs))
        return c

    def close(self):
        self.torch.cuda.synchronize(self.dev)
        for c in self._ctx.values():
            c.close()
        self._ctx = {}

    def set_data(self, g_host):
        self.g.copy_(self.torch.as_tensor(g_host, dtype=self.torch.float32))

    def set_steps(self, tau, sigma):
        self.tau, self.sigma = float(tau), float(sigma)
        for c in self._ctx.values():
            c.set_steps(self.tau, self.sigma)

    def reset(self, f0=None):
        for t in (self.f, self.ft, self.h2, self.h1):
            t.zero_()
        if f0 is not None:
            self.f.copy_(self.torch.as_tensor(f0, dtype=self.torch.float32))
            self.ft.copy_(self.f)

    def windows(self):
        """Temporal blocking: per slab the device window (w0, w1) of win_nz slices and its core (z0, z1).  After k <= block
        iterations of the CLOSED window the wrong boundary condition at an interior window end has spoiled k slices next to it
        (one per iteration: the dual step needs ft[z+1], the primal step h2_z[z-1]); the core keeps at least `block` slices of
        distance from every interior end, a window end at the volume's own boundary is exact."""
        out = []
        for z0, z1 in self.ranges:
            w0 = max(0, min(z0 - self.block, self.nz - self.win_nz))
            out.append((w0, w0 + self.win_nz, z0, z1))
        return out

    def _iterate_blocked(self, k):
        """k <= block iterations for the whole volume: every slab's window goes up from the current host copy, runs
        cp4d_iterate(k) (a CUDA-graph replay) as an ordinary closed volume, and its core comes down into the other host copy."""
        torch = self.torch
        Event = torch.cuda.Event
        cur = dict(f=self.f, ft=self.ft, h2=self.h2, h1=self.h1)
        nxt = self._nxt
        slot_free = [None] * self.depth
        for i, (w0, w1, z0, z1) in enumerate(self.windows()):
            slot = i % self.depth
            key = (slot, w1 - w0)
            if key not in self._ctx:
                self._ctx[key] = self._mk(w1 - w0, self.s_cmp[slot])
                self._ctx[key].set_steps(self.tau, self.sigma)
            c = self._ctx[key]
            st, cs = c.state(), self.s_cmp[slot]
            with torch.cuda.stream(self.s_in):
                if slot_free[slot] is not None:
                    self.s_in.wait_event(slot_free[slot])
                st["f"].copy_(cur["f"][w0:w1], non_blocking=True)
                st["ft"].copy_(cur["ft"][w0:w1], non_blocking=True)
                for a in range(4):
                    st["h2"][a].copy_(cur["h2"][a, w0:w1], non_blocking=True)
                st["h1"].copy_(cur["h1"][w0:w1], non_blocking=True)
                self.g_stage[slot][:w1 - w0].copy_(self.g[w0:w1], non_blocking=True)
                up = Event(); up.record(self.s_in)
            self.bytes_h2d += (w1 - w0) * (6 * self.n * self.n * self.mp + 2 * self.na * self.nd) * 4
            with torch.cuda.stream(cs):
                cs.wait_event(up)
                c.set_data(self.g_stage[slot][:w1 - w0])
                c.iterate(k)
                done = Event(); done.record(cs)
            a0, a1 = z0 - w0, z1 - w0
            with torch.cuda.stream(self.s_out):
                self.s_out.wait_event(done)
                nxt["f"][z0:z1].copy_(st["f"][a0:a1], non_blocking=True)
                nxt["ft"][z0:z1].copy_(st["ft"][a0:a1], non_blocking=True)
                for a in range(4):
                    nxt["h2"][a, z0:z1].copy_(st["h2"][a, a0:a1], non_blocking=True)
                nxt["h1"][z0:z1].copy_(st["h1"][a0:a1], non_blocking=True)
                fr = Event(); fr.record(self.s_out)
                slot_free[slot] = fr
            self.bytes_d2h += (z1 - z0) * (6 * self.n * self.n * self.mp + self.na * self.nd) * 4
        self.s_out.synchronize()
        self._nxt = cur
        self.f, self.ft, self.h2, self.h1 = nxt["f"], nxt["ft"], nxt["h2"], nxt["h1"]

    def iterate(self, n_iters):
        torch = self.torch
        if self.tau is None:
            raise binding.Cp4dError(binding.ESTATE, "set_steps first")
        if self.block > 1:
            left = n_iters
            while left > 0:
                k = min(self.block, left)
                self._iterate_blocked(k)
                left -= k
            return
        Event = torch.cuda.Event
        slot_free = [None] * self.depth                  # event: the slot's previous download has finished
        for _ in range(n_iters):
            h2z_ready = None                             # event: halo_h2z[(i-1) & 1] holds slab i-1's new last h2z slice
            for i, (z0, z1) in enumerate(self.ranges):
                slot = i % self.depth
                c = self._context(slot, i)
                st = c.state()
                cs = self.s_cmp[slot]
                # ---- host -> device (stream s_in): the slab's state and the OLD first ft slice of slab i+1 ----
                with torch.cuda.stream(self.s_in):
                    if slot_free[slot] is not None:
                        self.s_in.wait_event(slot_free[slot])
                    st["f"].copy_(self.f[z0:z1], non_blocking=True)
                    st["ft"].copy_(self.ft[z0:z1], non_blocking=True)
                    for a in range(4):                   # contiguous pieces: a strided host view would be staged through pageable memory
                        st["h2"][a].copy_(self.h2[a, z0:z1], non_blocking=True)
                    st["h1"].copy_(self.h1[z0:z1], non_blocking=True)
                    self.g_stage[slot][:z1 - z0].copy_(self.g[z0:z1], non_blocking=True)
                    if z1 < self.nz:
                        self.halo_ft[slot].copy_(self.ft[z1], non_blocking=True)
                    up = Event(); up.record(self.s_in)
                nb = (z1 - z0) * (6 * self.n * self.n * self.mp + 2 * self.na * self.nd) * 4
                self.bytes_h2d += nb + (self.n * self.n * self.mp * 4 if z1 < self.nz else 0)
                # ---- compute (the context's stream): dual + primal of this slab ----
                with torch.cuda.stream(cs):
                    cs.wait_event(up)
                    if h2z_ready is not None:
                        cs.wait_event(h2z_ready)
                    c.set_data(self.g_stage[slot][:z1 - z0])
                    c.step_dual(self.halo_ft[slot] if z1 < self.nz else None)
                    if z1 < self.nz:                     # keep the new last h2z slice for slab i+1 before the slot is reused
                        self.halo_h2z[i & 1].copy_(st["h2"][2, -1], non_blocking=True)
                    c.step_primal(self.halo_h2z[(i - 1) & 1] if i > 0 else None)
                    done = Event(); done.record(cs)
                    h2z_ready = done
                # ---- device -> host (stream s_out) ----
                with torch.cuda.stream(self.s_out):
                    self.s_out.wait_event(done)
                    self.f[z0:z1].copy_(st["f"], non_blocking=True)
                    self.ft[z0:z1].copy_(st["ft"], non_blocking=True)
                    for a in range(4):
                        self.h2[a, z0:z1].copy_(st["h2"][a], non_blocking=True)
                    self.h1[z0:z1].copy_(st["h1"], non_blocking=True)
                    fr = Event(); fr.record(self.s_out)
                    slot_free[slot] = fr
                self.bytes_d2h += (z1 - z0) * (6 * self.n * self.n * self.mp + self.na * self.nd) * 4
            # the next sweep reads ft[z1] of the host copy: every download of this sweep must have landed
            self.s_out.synchronize()

    def get_f(self):
        self.torch.cuda.synchronize(self.dev)
        return self.f


def exchange_halos(ft_first, h2z_last, ft_above, h2z_below, rank, world, phase, group=None):
    """Halo exchange between z-neighbours, one slab per rank (slab index = rank), as `torch.distributed` point-to-point pairs.

    phase "dual":   rank r sends its first ft slice DOWN to r-1 and receives r+1's into `ft_above`  (before cp4d_step_dual)
    phase "primal": rank r sends its last h2z slice UP to r+1 and receives r-1's into `h2z_below`   (before cp4d_step_primal)
    Tensors are one slice each, on the device of the backend (CUDA for nccl, CPU for gloo).  Returns after completion.
    """
    import torch.distributed as dist
    ops = []
    if phase == "dual":
        if rank > 0:
            ops.append(dist.P2POp(dist.isend, ft_first, rank - 1, group))
        if rank < world - 1:
            ops.append(dist.P2POp(dist.irecv, ft_above, rank + 1, group))
    elif phase == "primal":
        if rank < world - 1:
            ops.append(dist.P2POp(dist.isend, h2z_last, rank + 1, group))
        if rank > 0:
            ops.append(dist.P2POp(dist.irecv, h2z_below, rank - 1, group))
    else:
        raise ValueError(phase)
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()


def iterate_rank(slab, rank, world, n_iters, group=None):
    """Fig. 2 on one slab per rank with the two halo exchanges around the step calls.  `slab` provides one-slice tensors
    ft_first() / h2z_last() (views of its state), receive buffers ft_above / h2z_below, and step_dual(halo), step_primal(halo)."""
    for _ in range(n_iters):
        exchange_halos(slab.ft_first(), None, slab.ft_above, None, rank, world, "dual", group)
        slab.step_dual(slab.ft_above if rank < world - 1 else None)
        exchange_halos(None, slab.h2z_last(), None, slab.h2z_below, rank, world, "primal", group)
        slab.step_primal(slab.h2z_below if rank > 0 else None)


class RankSlab:
    """One slab per rank on that rank's GPU (slab index = rank); iterate with `iterate_rank(slab, rank, world, n)`."""

    def __init__(self, n, nz, nd, n_angles, n_half_rot, m, phi, rank, world, device=0, **kw):
        self.rank, self.world = rank, world
        self.z0, self.z1 = partition(nz, world)[rank]
        self.ctx = binding.Context(n, self.z1 - self.z0, nd, n_angles, n_half_rot, m, phi, device=device,
                                   z_open=z_open_flags(rank, world), **kw)
        self.st = self.ctx.state()
        t = self.ctx.torch
        shape = self.st["ft"][0].shape
        self.ft_above = t.empty(shape, dtype=t.float32, device=self.ctx.device)
        self.h2z_below = t.empty(shape, dtype=t.float32, device=self.ctx.device)
        self.step_dual, self.step_primal = self.ctx.step_dual, self.ctx.step_primal

    def ft_first(self):
        return self.st["ft"][0]

    def h2z_last(self):
        return self.st["h2"][2, -1]
