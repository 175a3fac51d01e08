"""Host logic of bench.py's N > 1 path ("replicas only") with world_size 2 over gloo on the CPU:
the per-rank times are reduced with MAX and the whole-job value is all ranks' steps over the slowest rank's time."""
import os
import socket
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, str(ROOT))
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
    ms_max = bench.reduce_max(ms, world, "cpu")
    dist.barrier()
    out.put((rank, ms_max, bench.replicas_value(world, 4, ms_max)))
    dist.destroy_process_group()


def test_replicas_max_over_ranks_gloo():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms_max, val in res:
        assert ms_max == 15.0
        assert val == pytest.approx(2 * 4 / 15e-3)


def test_single_rank_is_identity():
    sys.path.insert(0, str(ROOT))
    import bench
    assert bench.reduce_max(3.5, 1) == 3.5
    assert bench.replicas_value(1, 10, 100.0) == pytest.approx(100.0)


def test_json_line_contract_offline():
    """bench.assemble on a canned run record: the keys and invariants of the bench contract (no GPU needed)."""
    sys.path.insert(0, str(ROOT))
    import bench
    from paper_1809_09725_b200 import synth

    class A:
        steps, warmup, frames, projectors = 50, 5, 0, "auto"
    c = synth.CONFIGS[3]
    prof = {k: (ms * 50, 50) for k, ms in dict(forward=6.7, backproject=3.8, prox_f2=0.76, update=0.61, synth=0.09, fold=0.07).items()}
    r = dict(ms=600.0, launches=350, prof=prof, prof_gd={"grad": (1.38, 3), "div": (1.2, 3)}, ops={"forward_op": 6.7, "adjoint_op": 3.85},
             e2e={"value": 81.0, "unit": bench.UNIT, "h2d_bytes_per_step": 1.0, "d2h_bytes_per_step": 2.0},
             clocks={"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "reasons": []}, peaks=bench.load_peaks(), L=1.0, launches_total=1,
             graph_replays=55, fp32_alt=None, proj=("tensor", "tensor"), step="two-kernel")
    line = bench.assemble(A, c, 1, r)
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "roofline", "e2e", "clocks", "gpu_launches"):
        assert k in line, k
    assert line["value"] == pytest.approx(50 / 0.6) and line["ms_per_step"] == pytest.approx(12.0)
    assert line["dtype"] == "f32" and line["data"] == "synthetic" and line["vs_baseline"] is None and line["scaling"] == "weak"
    assert "workload" in line["config"] and "model" not in line["config"]
    rf = line["roofline"]
    assert rf["kernel"] == "forward" and rf["bound"] == "alu" and rf["unit"] == "TFLOP/s"
    assert rf["frac"] == pytest.approx(rf["achieved"] / rf["peak"]) and 0 < rf["frac"] < 1
    # algorithmic flops of the forward kernel: 2 flop x 2 taps x m x N^2 Nz N_theta0
    assert rf["achieved"] * 1e12 * 6.7e-3 == pytest.approx(2 * 2 * c.m * c.n ** 2 * c.nz * c.n_theta0, rel=1e-9)
    # tensor-core forward kernel: 12 dense-equivalent MACs per algorithmic FMA against the measured rate of the 2:4 sparse
    # mma.sp.m16n8k32, 16 x 8 x 32 per 9.71 clk and sub-partition (profiles/r2_microbench.md)
    per_clk = 4 * 16 * 8 * 32 / 9.71
    assert rf["second_roof"]["frac"] == pytest.approx(rf["achieved"] / 2 * 12 / (148 * per_clk * r["peaks"]["sm_max_mhz"] * 1e6 / 1e12), rel=1e-6)
    assert line["run"]["projectors"] == {"mode": "auto", "forward": "tensor", "adjoint": "tensor"}
    r2 = dict(r, proj=("fp32", "fp32"))
    rf2 = bench.assemble(A, c, 1, r2)["roofline"]
    assert rf2["second_roof"]["frac"] == pytest.approx(4 * rf2["frac"] * (148 * 128 * 2 * r["peaks"]["sm_max_mhz"] * 1e6 / 1e12) / rf2["peak"], rel=1e-6)
    hbm = line["kernels"]["prox_f2"]
    assert hbm["bound"] == "hbm" and hbm["achieved"] == pytest.approx(9 * c.V * 4 / 0.76e-3 / 1e9)


def _run_bench(argv, env_extra=None):
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    env.update(env_extra or {})
    return subprocess.run([sys.executable, str(ROOT / "bench.py"), *argv], env=env, capture_output=True, text=True, timeout=300)


def test_gpus_n_without_enough_devices_exits_nonzero():
    """`python bench.py --gpus N` starts N ranks itself; with fewer than N CUDA devices it must refuse, not print an N = 1 line."""
    import torch
    if torch.cuda.device_count() >= 2:
        pytest.skip("box has >= 2 GPUs")
    r = _run_bench(["--gpus", "2", "--steps", "1"])
    assert r.returncode != 0 and r.stdout.strip() == "" and "--gpus 2" in r.stderr


def test_gpus_n_disagreeing_with_world_size_exits_nonzero():
    r = _run_bench(["--gpus", "2", "--steps", "1"], {"WORLD_SIZE": "4", "RANK": "0"})
    assert r.returncode != 0 and r.stdout.strip() == "" and "WORLD_SIZE=4" in r.stderr


def test_traffic_is_tied_to_the_kernel_sources():
    """profiles/traffic.json carries the SHA-1 of csrc/ it was captured with; bench.py reports its numbers only on a match."""
    import json
    sys.path.insert(0, str(ROOT))
    import bench
    sha = bench.csrc_sha1()
    assert len(sha) == 40 and sha == bench.csrc_sha1()
    tj = json.loads((ROOT / "profiles" / "traffic.json").read_text())
    assert "csrc_sha1" in tj
