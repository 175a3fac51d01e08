#!/usr/bin/env python
"""bench.py -- one JSON line per run: CP iterations/s of the cp4d hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl cp4d|reference]

A "step" is ONE Chambolle-Pock iteration (Fig. 2: forward + F1* prox, grad + F2* prox,
adjoint, div + primal update + over-relaxation) over the whole 4D problem of `--config` (BASELINE.json configs,
numbered 1..5 as in SURVEY.md 8).  Inputs are seeded and synthetic (paper_1809_09725_b200/synth.py; DESIGN.md
"Input recipe"); the iteration's cost does not depend on the values.

  value    : iterations/s, state resident in HBM, K iterations enqueued by cp4d_iterate, CUDA events on the
             context's stream, barrier + synchronize on both sides, max over ranks.
  e2e      : the same metric through cp4d_solve_host(g_host, K, f_host): pinned HOST buffers, H2D of the
             sinogram, reset, K iterations, D2H of f, all inside the timed region.
  roofline : the dominant kernel of the step (largest share of device time in the timed region), timed live
             by the library's per-kernel CUDA events (cp4d_profile_begin/end) during a second pass of K steps.
  kernels  : the same for every kernel class, plus nominal voxel*angle*basis GUPS of forward and adjoint.
  cpu_baseline : the fp64 oracle (oracle/cp4d_ref.c, as it stands) on this box's host cores, on a bounded
             sample (a few full in-plane slices), extrapolated to the whole problem.

The default workload is config 5 (2048^2 x 32, 3600 angles, m = 16: the largest single-GPU configuration of BASELINE.json,
110 GB of workspace with the one-pass step of `--step one-pass`, the default; 67 GB with `--step two-kernel`); `--config 3` is
the quick one.

N > 1: the path does not shard (north_star: one GPU); `--gpus N` runs N independent replicas, one per rank,
no data-path collective ("replicas only"): the value is REPLICA throughput.  Started without a
launcher (`python bench.py --gpus N`, no WORLD_SIZE in the environment) it re-executes itself under
`python -m torch.distributed.run --nproc-per-node N`; if the box has fewer than N GPUs, or WORLD_SIZE disagrees with N,
it exits non-zero instead of printing a line for fewer GPUs.  `--impl reference` times the oracle only.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import socket
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "cp_iterations_per_s"
UNIT = "it/s"
N_SM, LANES = 148, 128


def load_peaks():
    """Roofline denominators: MEASURED_PEAKS.json (driver-written) else the profiling guide's fallback."""
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


def csrc_sha1() -> str:
    """SHA-1 over the kernel sources: profiles/traffic.json stores the one its ncu capture was taken with, and its DRAM bytes
    are only reported for the kernels that are actually running (a stale capture gives "traffic": null)."""
    h = hashlib.sha1()
    d = ROOT / "paper_1809_09725_b200" / "csrc"
    for f in sorted(list(d.glob("*.cu")) + list(d.glob("*.cuh"))):
        h.update(f.name.encode())
        h.update(f.read_bytes())
    return h.hexdigest()


def alu_peak_tflops(sm_mhz: float) -> float:
    """Plain FP32 FMA pipe: 148 SMs x 128 lanes x 2 flop x clock."""
    return N_SM * LANES * 2 * sm_mhz * 1e6 / 1e12


# ------------------------------------------------------------------------------------------------------
# algorithmic work per launch of each kernel class (bytes or flops per unit x units)
# ------------------------------------------------------------------------------------------------------
def algorithmic_work(c, n_frames=0):
    V, S = c.V, c.S
    n0 = c.n_theta0
    mproj = c.m                                          # images the projector pair carries per voxel
    Vc = V                                               # coefficient stack (K1 o A path)
    if n_frames:
        V = V // c.m * n_frames                          # primal arrays hold frames
        if n_frames <= c.m:                              # collapsed frame mode: the projectors carry the N_t frames
            mproj, Vc = n_frames, 0
    ray_fma = 2 * mproj * c.n * c.n * c.nz * n0          # 2 taps x images per voxel-step per base-angle ray
    syn_fma = mproj * c.n_angles * c.nd * c.nz           # synthesis / analysis per sinogram sample
    gt = c.nz * n0 * c.nd * mproj                        # folded sinogram / partial ray sums, elements
    return {
        # name: (bound, work per launch [flop or byte])
        # both projectors are rated against the plain FP32 FMA roof on their ALGORITHMIC flops, whichever pipe runs them (the
        # tensor-core forward kernel executes 12 x as many MACs on the HMMA pipe to deliver these)
        "forward": ("alu", 2.0 * ray_fma),
        "backproject": ("alu", 2.0 * ray_fma),
        "synth": ("hbm", 4.0 * (gt + 3 * S)),            # read P, read h1 + g, write h1 (prox fused)
        "fold": ("hbm", 4.0 * (S + gt)),
        "grad": ("hbm", 4.0 * 5 * V),
        "div": ("hbm", 4.0 * 5 * V),
        "prox_f2": ("hbm", 4.0 * 9 * V),                 # read ft + h2[4], write h2[4]
        "update": ("hbm", 4.0 * 8 * V),                  # read h2[4] + f + K1^T h1, write f + ft
        "prox_update": ("hbm", 4.0 * 13 * V),            # the two in one pass: read ft + h2[4] + f + K1^T h1, write h2[4] + f + ft
        "mix": ("hbm", 4.0 * (V + Vc)),                  # frame mode: read frames / write coefficients or the reverse
    }


def reduce_max(value: float, world: int, device="cpu") -> float:
    """MAX over ranks of a per-rank time (the contract: multi-GPU numbers are the slowest rank's).  Uses the
    initialised torch.distributed group (nccl on GPU boxes, gloo in the CPU tests); identity when world == 1."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replicas_value(world: int, steps: int, ms_max: float) -> float:
    """Whole-job it/s of `world` independent replicas ("replicas only"): all ranks' steps / slowest rank's time."""
    return world * steps / (ms_max * 1e-3)


class ClockSampler:
    """nvidia-smi clocks + throttle reasons every 200 ms during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, uuid: str | None):
        self.rows, self.proc = [], None
        cmd = ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200"]
        if uuid:
            cmd += ["-i", uuid]
        try:
            self.proc = subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [x.strip() for x in line.split(",")]))

    def mark(self):
        return time.perf_counter()

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        rows = [r for t, r in self.rows if t0 <= t <= t1 + 0.2] or [r for _, r in self.rows]
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------------
# CPU baseline / reference arm: the fp64 oracle as it stands, on a bounded sample of the same workload
# ------------------------------------------------------------------------------------------------------
def oracle_sample_config(c, target_fma: float = 4e10):
    """A sub-problem with the full in-plane size, angles and basis but only nz_s of the nz slices.
    K1/K1^T and the proxes are independent per slice and the stencils cost the same per element, so one CP
    iteration of the sub-problem x (nz/nz_s) is one CP iteration of the workload."""
    per_slice = 4.0 * c.m * c.n * c.n * c.n_theta0          # forward + adjoint FMA of one slice, folded
    nz_s = int(max(1, min(c.nz, round(target_fma / per_slice))))
    return c.scaled(nz=nz_s), c.nz / nz_s


def oracle_steps(c, steps: int, warmup: int, target_fma: float = 4e10, n_frames: int = 0):
    """Times `steps` oracle CP iterations (all host cores, pi-folded operators -- bitwise equal to 1 thread)
    on the sample; returns (it/s extrapolated to the workload, cores, sample text, seconds per sample step)."""
    from oracle import ref
    from paper_1809_09725_b200 import synth
    ref.build()
    cores = ref.max_threads()
    ref.set_threads(cores)
    cs, scale = oracle_sample_config(c, target_fma)
    phi = synth.basis_table(cs.basis, cs.m, cs.n_angles)
    if n_frames:
        P = ref.FrameProblem(cs.n, cs.nz, cs.nd, cs.n_angles, cs.n_half_rot, cs.m, phi, n_frames, cs.lambda1, cs.lambda2)
    else:
        P = ref.Problem.from_config(cs, phi=phi)
    r = synth.rng(c.cfg, 1)
    g = r.standard_normal(P.sino_shape)                      # cost does not depend on the values
    st = P.zero_state()
    st["ft"][:] = r.standard_normal(P.primal_shape)
    ts = 0.01
    for _ in range(warmup):
        P.cp(g, st, ts, ts, 1, folded=True)
    t0 = time.perf_counter()
    for _ in range(steps):
        P.cp(g, st, ts, ts, 1, folded=True)
    dt = (time.perf_counter() - t0) / max(steps, 1)
    ref.set_threads(1)
    sample = (f"{steps} oracle CP iteration(s) (fp64, pi-folded, OpenMP over outputs) on {cs.nz} of {c.nz} slices at full "
              f"in-plane size {c.n}x{c.n}, {c.n_angles} angles, m={c.m}; x{scale:g} slices")
    return 1.0 / (dt * scale), cores, sample, dt


def workload_config(c, n_frames=0):
    """The `config` object both arms print (same keys, so the driver can tell they ran the same workload)."""
    from paper_1809_09725_b200 import synth
    return {"workload": synth.describe(c) + (f"_frames{n_frames}" if n_frames else ""), "n_frames": n_frames, "cfg": c.cfg,
            "n": c.n, "nz": c.nz, "nd": c.nd, "n_angles": c.n_angles, "n_half_rot": c.n_half_rot, "m": c.m, "basis": c.basis,
            "lambda1": c.lambda1, "lambda2": c.lambda2}


def run_reference(args, c, rank):
    """--impl reference: the oracle on the host cores (rank 0 only), same metric/config as our arm."""
    if rank != 0:
        return
    from paper_1809_09725_b200 import synth
    # every step is one oracle CP iteration on a bounded slice sample (one slice at configs 4-5); W untimed + K timed steps
    val, cores, sample, dt = oracle_steps(c, args.steps, min(args.warmup, 1), target_fma=1.5e10, n_frames=args.frames)
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(c, args.frames),
        "note": ("fp64 CPU oracle (oracle/cp4d_ref.c): ms_per_step is the measured time of one step on the slice sample; value is "
                 "the whole-workload it/s, i.e. 1 / (ms_per_step x slices / sample slices)"),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                         "sample_step_s": dt},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------------
def run_cp4d(args, c, rank, world):
    import torch
    import torch.distributed as dist
    from paper_1809_09725_b200 import binding, build, synth

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the cp4d hot path has no CPU fallback")
    local = int(os.environ.get("LOCAL_RANK", rank))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    # everything runs on one non-default stream: cp4d_iterate replays a CUDA graph of one iteration there (the legacy
    # default stream cannot be captured); the CUDA events below are recorded on this same stream
    torch.cuda.set_stream(torch.cuda.Stream(dev))
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    if rank == 0:
        build.build_lib()
    if world > 1:
        dist.barrier()
    peaks = load_peaks()
    K, W = args.steps, max(args.warmup, 2)     # >= 2: the CUDA graph of one iteration is captured and instantiated in the warm-up

    # ---- problem, data, step sizes (outside the timed region: SURVEY 8(d)) ----
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    # --step one-pass: the workspace holds second copies of h2 and ft, and cp4d_iterate runs steps 4-6 as one kernel
    ctx = binding.Context.from_config(c, phi=phi, device=local, n_frames=args.frames, fused=args.step == "one-pass")
    ctx.set_projector_mode(args.projectors)
    g = synth.sinogram(c, device=str(dev)).to(torch.float32).contiguous()
    L = ctx.norm(args.power_iters, seed=3)
    ts = 0.95 / L
    ctx.set_steps(ts, ts)
    ctx.set_data(g)
    ctx.reset()
    launches0 = ctx.launch_count()

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize(dev)

    # ---- value: K iterations, state resident in HBM ----
    ctx.iterate(W)
    uuid = None
    try:
        uuid = "GPU-" + str(torch.cuda.get_device_properties(dev).uuid).replace("GPU-", "")
    except Exception:
        pass
    sampler = ClockSampler(uuid)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = ctx.launch_count()
    t0 = sampler.mark()
    e0.record(ctx.stream)
    ctx.iterate(K)
    e1.record(ctx.stream)
    barrier()
    t1 = sampler.mark()
    launches = ctx.launch_count() - l0
    ms = e0.elapsed_time(e1)
    graph_replays = ctx.graph_replays()

    # ---- the same K steps with the fp32 CUDA-core kernels on both sides (context only: the default pair uses split-bf16
    # tensor-core products in the forward projector; both pass the same parity tests) ----
    fp32_alt = None
    if args.projectors == "auto" and ctx.projector_mode_in_use() != ("fp32", "fp32"):
        ctx.set_projector_mode("fp32")
        ctx.iterate(2)
        barrier()
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record(ctx.stream); ctx.iterate(K); a1.record(ctx.stream)
        barrier()
        ms_alt = reduce_max(a0.elapsed_time(a1), world, dev)
        fp32_alt = {"value": replicas_value(world, K, ms_alt), "unit": UNIT, "ms_per_step": ms_alt / K,
                    "note": "same K steps with cp4d_set_projector_mode(CP4D_PROJ_FP32): plain fp32 FMAs in both projectors"}
        ctx.set_projector_mode("auto")
        ctx.iterate(2)

    # ---- roofline: second pass of K steps with the library's per-kernel CUDA events on the same stream ----
    ctx.profile_begin()
    ctx.iterate(K)
    prof = ctx.profile_end()
    clocks = sampler.stop(t0, time.perf_counter())
    ms = reduce_max(ms, world, dev)

    # ---- standalone operators (grad/div are not launched by the fused iteration) ----
    f_t, g_t = ctx.empty_primal().normal_(), ctx.empty_sino().normal_()
    p_t = ctx.empty_dual()
    ctx.profile_begin()
    for _ in range(3):
        ctx.grad(f_t, out=p_t)
        ctx.div(p_t, out=f_t)
    prof_gd = ctx.profile_end()
    del p_t
    ops = {}
    for name, fn in (("forward_op", lambda: ctx.forward(f_t, out=g_t)), ("adjoint_op", lambda: ctx.adjoint(g_t, out=f_t))):
        fn()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        tt = []
        for _ in range(3):
            a.record(ctx.stream); fn(); b.record(ctx.stream); b.synchronize()
            tt.append(a.elapsed_time(b))
        ops[name] = float(np.median(tt))
    del f_t, g_t

    # ---- e2e: cp4d_solve_host with pinned HOST buffers, copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        g_host = g.cpu().pin_memory()
        f_host = torch.empty(ctx.primal_shape, dtype=torch.float32).pin_memory()
        ctx.solve_host(g_host, 1, f_host)                 # warm the copy paths
        barrier()
        w0 = time.perf_counter()
        ctx.solve_host(g_host, K, f_host)                 # syncs before returning
        w1 = time.perf_counter()
        dt = w1 - w0
        dt = reduce_max(dt, world, dev)
        e2e = {"value": world * K / dt, "unit": UNIT, "h2d_bytes_per_step": c.S * 4 / K, "d2h_bytes_per_step": c.V * 4 / K,
               "call": f"cp4d_solve_host(g_host, {K}, f_host): H2D {c.S * 4} B + reset + {K} iterations + D2H {c.V * 4} B, pinned host memory",
               "seconds": dt}
        del g_host, f_host
    return ctx, dict(ms=ms, launches=launches, prof=prof, prof_gd=prof_gd, ops=ops, e2e=e2e, clocks=clocks, peaks=peaks,
                     fp32_alt=fp32_alt, proj=ctx.projector_mode_in_use(), step="one-pass" if ctx.fused_step_in_use() else "two-kernel",
                     L=L, launches_total=ctx.launch_count() - launches0, graph_replays=graph_replays)


def run_streamed(args, c, L):
    """Out-of-core variant: the CP state stays in pinned host memory and passes through the
    GPU slab by slab every iteration, copies on their own streams.  Wall-clock over K iterations after one warm-up sweep."""
    import torch
    from paper_1809_09725_b200 import slabs, synth
    phi = synth.basis_table(c.basis, c.m, c.n_angles)
    T = slabs.StreamedSolver(c.n, c.nz, c.nd, c.n_angles, c.n_half_rot, c.m, phi, slab_nz=args.streamed, n_frames=args.frames,
                             block=args.stream_block, lambda1=c.lambda1, lambda2=c.lambda2)
    T.set_data(synth.sinogram(c).to(torch.float32))
    T.set_steps(0.95 / L, 0.95 / L)
    T.reset()
    T.iterate(max(1, min(args.warmup, 2)) * args.stream_block)
    torch.cuda.synchronize()
    K = max(2, args.steps // 5) * args.stream_block
    b0, d0 = T.bytes_h2d, T.bytes_d2h
    t0 = time.perf_counter()
    T.iterate(K)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    h2d, d2h = (T.bytes_h2d - b0) / K, (T.bytes_d2h - d0) / K
    out = {"value": K / dt, "unit": UNIT, "steps": K, "slab_nz": args.streamed, "slabs": T.n_slabs, "device_contexts": T.depth,
           "block": args.stream_block, "window_nz": T.win_nz if args.stream_block > 1 else args.streamed,
           "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "h2d_gbs": h2d * K / dt / 1e9, "d2h_gbs": d2h * K / dt / 1e9,
           "note": "state (f, ft, h2, h1, g) in pinned host memory; every iteration streams it through the GPU once"}
    T.close()
    return out


def assemble(args, c, world, r):
    from paper_1809_09725_b200 import synth
    peaks, K = r["peaks"], args.steps
    work = algorithmic_work(c, args.frames)
    alu_peak = alu_peak_tflops(peaks["sm_max_mhz"])
    kernels, total_ms = {}, 0.0
    merged = dict(r["prof"])
    merged.update({k: v for k, v in r["prof_gd"].items() if k in ("grad", "div")})
    for name, (ms_sum, n) in merged.items():
        if name not in work or not n:
            continue
        bound, w = work[name]
        avg = ms_sum / n
        if bound == "alu":
            ach, peak, unit = w / (avg * 1e-3) / 1e12, alu_peak, "TFLOP/s"
        else:
            ach, peak, unit = w / (avg * 1e-3) / 1e9, peaks["hbm_gbs"], "GB/s"
        kernels[name] = {"bound": bound, "achieved": ach, "peak": peak, "unit": unit, "frac": ach / peak, "ms": avg,
                         "launches": n, "in_step": name in r["prof"]}
        if name in r["prof"]:
            total_ms += ms_sum
    for name, k in kernels.items():
        k["share_of_step"] = (k["ms"] * k["launches"] / total_ms) if (k["in_step"] and total_ms) else None
    dom = max((n for n in kernels if kernels[n]["in_step"]), key=lambda n: kernels[n]["ms"] * kernels[n]["launches"])
    d = kernels[dom]
    roofline = {"kernel": dom, "bound": d["bound"], "achieved": d["achieved"], "peak": d["peak"], "unit": d["unit"],
                "frac": d["frac"], "traffic": None, "peak_source": peaks["source"], "avg_launch_ms": d["ms"],
                "note": ("alu peak = 148 SM x 128 FP32 lanes x 2 flop x sm_max_mhz; achieved = algorithmic (pi-folded) flops"
                         if d["bound"] == "alu" else "algorithmic bytes / CUDA-event time")}
    # second, tighter roofs of the forward projector (measured unit rates in profiles/r2_microbench.md):
    #   fp32 gather: one 4-byte operand per FMA through shared memory, 128 B/clk/SM;
    #   tensor-core kernel: every algorithmic FMA costs 12 dense-equivalent MACs (weight blocks 1/4 dense x three split-bf16
    #   products); the 2:4 sparse mma.sp.m16n8k32 takes 16 x 8 x 32 of them per 9.71 clk and sub-partition (measured), i.e.
    #   1687 dense-equivalent MAC/clk/SM.
    if "forward" in kernels:
        k = kernels["forward"]
        fmas = work["forward"][1] / 2.0
        if r["proj"][0] == "tensor":
            per_clk = 4 * 16 * 8 * 32 / 9.71
            peak = N_SM * per_clk * peaks["sm_max_mhz"] * 1e6 / 1e12
            ach = fmas * 12.0 / (k["ms"] * 1e-3) / 1e12
            k["hmma_roof"] = {"bound": "tensor (mma.sp 2:4)", "achieved": ach, "peak": peak, "unit": "TMAC/s", "frac": ach / peak,
                              "note": "12 dense-equivalent MACs per algorithmic FMA (not counting partly filled blocks); peak = 148 SM x 4 x "
                                      "16*8*32 MAC per 9.71 clk (HMMA.SP.16832, measured) x sm_max_mhz"}
        else:
            smem_peak = N_SM * 128 * peaks["sm_max_mhz"] * 1e6 / 1e9                       # GB/s
            smem_ach = fmas * 4.0 / (k["ms"] * 1e-3) / 1e9
            k["smem_roof"] = {"bound": "smem", "achieved": smem_ach, "peak": smem_peak, "unit": "GB/s", "frac": smem_ach / smem_peak,
                              "note": "one 4-byte operand per FMA through shared memory: 148 SM x 128 B/clk x sm_max_mhz"}
        if dom == "forward":
            roofline["second_roof"] = k.get("hmma_roof") or k.get("smem_roof")
    # dram bytes per launch from the committed `ncu --set full` capture -- only if it was taken with the kernel sources that
    # are running now (profiles/traffic.json records their SHA-1); otherwise null, never a stale number
    tr = ROOT / "profiles" / "traffic.json"
    roofline["traffic_source"] = None
    if tr.exists():
        try:
            tj = json.loads(tr.read_text())
            if tj.get("csrc_sha1") == csrc_sha1():
                per_kernel = tj.get(synth.describe(c), {})
                roofline["traffic"] = per_kernel.get(dom)
                roofline["traffic_source"] = f"profiles/traffic.json (ncu --set full, csrc sha1 {tj['csrc_sha1'][:12]})"
                for n, k in kernels.items():
                    k["traffic"] = per_kernel.get(n)
            else:
                roofline["traffic_source"] = "profiles/traffic.json is from other kernel sources: not reported"
        except Exception:
            pass
    gups = {n: c.nominal_updates / (r["ops"][n + "_op"] * 1e-3) / 1e9 for n in ("forward", "adjoint")}
    ms_step = r["ms"] / K
    line = {
        "metric": METRIC, "value": replicas_value(world, K, r["ms"]), "unit": UNIT, "n_gpus": world, "steps": K,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": workload_config(c, args.frames),
        "run": {"norm_K": r["L"], "projectors": {"mode": args.projectors, "forward": r["proj"][0], "adjoint": r["proj"][1]},
                "step": r["step"],
                "arithmetic": ("fp32 storage, fp32 accumulation everywhere; 'tensor' projector = products of split-bf16 pairs "
                               "(x = hi + lo, three products per term on the 2:4 sparse mma.sp, rel. error 5e-6 per ray sum or voxel, tolerance 1e-4), "
                               "'fp32' projector = plain FMAs (2e-6)"), "parallelism": "replicas only (independent problems, no collective)" if world > 1 else "1 gpu",
                "warmup_run": max(args.warmup, 2),
                "l2": f"no flush: CP state {(7 * c.V + 2 * c.S) * 4 / 1e9:.2f} GB streams through every step (L2 = 126 MB)"},
        "gups_nominal": {"forward": gups["forward"], "adjoint": gups["adjoint"], "unit": "1e9 voxel*angle*basis/s",
                         "forward_ms": r["ops"]["forward_op"], "adjoint_ms": r["ops"]["adjoint_op"],
                         "note": "nominal count N^2*Nz*N_theta*m per call; kernels use the pi-fold (N_theta0 base angles)"},
        "roofline": roofline, "kernels": kernels, "clocks": r["clocks"], "e2e": r["e2e"],
        "fp32_projectors": r["fp32_alt"],
        "gpu_launches": r["launches"], "cuda_graph_replays": r["graph_replays"], "impl": "cp4d",
    }
    return line


def spawn_ranks(n: int) -> int:
    """`python bench.py --gpus N` without a launcher: re-execute under torch.distributed.run, one rank per GPU (the command the
    driver itself uses for N > 1).  Returns the launcher's exit code; refuses (non-zero) when the box has fewer GPUs."""
    import torch
    have = torch.cuda.device_count()
    if have < n:
        print(f"bench.py: --gpus {n} but only {have} CUDA device(s) visible: not printing a line for fewer GPUs", file=sys.stderr)
        return 2
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), str(Path(__file__).resolve()), *sys.argv[1:]]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=5,
                    help="BASELINE.json config 1..5 (SURVEY.md 8 numbering); default 5 = the largest single-GPU config, 3 = quick")
    ap.add_argument("--impl", default="cp4d", choices=["cp4d", "reference"])
    ap.add_argument("--power-iters", type=int, default=30, help="power-iteration steps for ||K|| (DESIGN.md R8: 30)")
    ap.add_argument("--frames", type=int, default=0, help="N_t > 0: the paper's frame discretisation (cp4d_params.n_frames), e.g. 8")
    ap.add_argument("--streamed", type=int, default=0, metavar="SLAB_NZ",
                    help="also time the out-of-core path (slabs.StreamedSolver: state in pinned host memory, slabs of SLAB_NZ slices)")
    ap.add_argument("--stream-block", type=int, default=1, metavar="K",
                    help="with --streamed: temporal blocking, K iterations per residency of a window of SLAB_NZ + 2K slices")
    ap.add_argument("--projectors", default="auto", choices=["auto", "fp32", "tensor"],
                    help="cp4d_set_projector_mode: auto = the tensor-core pair where the problem fills the GPU, else the fp32 kernels "
                         "(default); fp32 = CUDA-core kernels on both sides; tensor = tensor-core kernels on both sides")
    ap.add_argument("--step", default="one-pass", choices=["one-pass", "two-kernel"],
                    help="one-pass (default): workspace of cp4d_workspace_bytes_fused, steps 4-6 of Fig. 2 in one kernel (13 V floats of "
                         "HBM traffic); two-kernel: the smaller workspace, prox and update as two kernels (17 V)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    from paper_1809_09725_b200 import synth
    c = synth.CONFIGS[args.config]
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    if args.impl == "reference":                       # the oracle on the host cores: rank 0 alone works, whatever N is
        run_reference(args, c, rank)
        return
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        sys.exit(spawn_ranks(args.gpus))               # no launcher: start N ranks ourselves, one replica per GPU
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: refusing to print a line for another GPU count")
    import torch
    if torch.cuda.device_count() < int(os.environ.get("LOCAL_WORLD_SIZE", world)):
        raise SystemExit(f"bench.py: {world} ranks but only {torch.cuda.device_count()} CUDA device(s) visible")
    if args.warmup < 3:
        print(f"bench.py: warning: --warmup {args.warmup} < 3 (timing rules want >= 3)", file=sys.stderr)
    ctx, r = run_cp4d(args, c, rank, world)
    ctx.close()
    streamed = run_streamed(args, c, r["L"]) if (args.streamed and world == 1) else None
    if rank == 0:
        line = assemble(args, c, world, r)
        if streamed:
            line["streamed"] = streamed
        if not args.no_cpu_baseline and world == 1:
            val, cores, sample, dt = oracle_steps(c, 1, 0, target_fma=1.2e11, n_frames=args.frames)   # about 10 s of oracle work on 16 cores
            line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                                    "sample_step_s": dt}
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
