"""CPU tests of the host-side pieces around the hot path: the routing-trace dump and the
multi-rank contract of bench.py (replicas only): gloo world_size 2, rank 0 alone prints."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

import workloads as wl
from oracle import moe_oracle as orc
from paper_2605_31463_b200 import trace

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_routing_trace_schema_and_validity(tmp_path):
    layers = []
    for cfg in (wl.QWEN3_SMALL, wl.DSV3_SMALL.replace(routed_scale=1.0)):
        idx, w = orc.route(wl.gen_logits(cfg), wl.gen_bias(cfg), cfg)
        layers.append((idx.astype(np.int32), w.astype(np.float32)))
    p = trace.dump_routing_trace(str(tmp_path), 3, layers[:1])
    assert os.path.basename(p) == "step-00000003.npz"
    assert trace.check_routing_trace(p, wl.QWEN3_SMALL.E) == 1
    z = np.load(p)
    assert z["layer0.expert_ids"].shape == (wl.QWEN3_SMALL.T, wl.QWEN3_SMALL.K)
    assert z["layer0.gating_weights"].dtype == np.float32
    p2 = trace.dump_routing_trace(str(tmp_path), 4, layers[1:])
    assert trace.check_routing_trace(p2, wl.DSV3_SMALL.E) == 1
    with pytest.raises(ValueError):
        trace.check_routing_trace(p, 3)                       # IDs out of range for a 3-expert model
    bad = (layers[0][0], layers[0][1] * 0.5)
    with pytest.raises(ValueError):
        trace.check_routing_trace(trace.dump_routing_trace(str(tmp_path), 5, [bad]), wl.QWEN3_SMALL.E)


def _run(cmd, env=None):
    e = dict(os.environ)
    e.update(env or {})
    return subprocess.run(cmd, cwd=ROOT, env=e, capture_output=True, text=True, timeout=600)


def test_bench_reference_arm_single_process():
    r = _run([sys.executable, "bench.py", "--impl", "reference", "--steps", "1", "--warmup", "0", "--config", "tiny_fp32"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["config"]["workload"] == "tiny_fp32"


def test_bench_reference_arm_two_ranks_rank0_prints():
    """Launched as the driver does for N > 1 (torch.distributed.run, 127.0.0.1): rank 0 alone runs and prints."""
    r = _run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
              "127.0.0.1", "--master-port", "29611", "bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1",
              "--warmup", "0", "--config", "tiny_fp32"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1 and json.loads(lines[0])["n_gpus"] == 2


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, device="cpu")     # rank 1 is the slow replica
    seeds = bench.replica_seed(wl.TINY, rank).seed
    q.put((rank, ms, seeds))
    dist.destroy_process_group()


def test_replica_timing_is_max_over_ranks_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, 29613, q)) for r in range(2)]
    for p in ps:
        p.start()
    got = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
    assert [g[1] for g in got] == [15.0, 15.0]               # every rank sees the slowest replica's time
    assert got[0][2] != got[1][2]                            # each replica draws its own batch


def test_ncu_summary_parses_raw_and_launch_csv(tmp_path):
    """The script that writes profiles/*.md and profiles/traffic.json (bench.py's roofline.traffic) from ncu CSV exports:
    unit scaling, kernel naming, and the per-stage traffic (wgrad = mean of its three heaviest launches)."""
    import json
    import ncu_summary
    hdr = ["ID", "Kernel Name", "gpu__time_duration.sum", "dram__bytes_read.sum", "dram__bytes_write.sum",
           "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "lts__throughput.avg.pct_of_peak_sustained_elapsed",
           "sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active", "launch__registers_per_thread", "launch__grid_size"]
    units = ["", "", "us", "Mbyte", "Gbyte", "%", "%", "%", "register/thread", ""]
    k = "void moe::(anonymous namespace)::tc_gemm_kernel<%d, %d, 0>(CUtensorMap_st, TcParams)"
    rows = [[str(i), k % (m, pr), t, rd, wr, "50", "40", "60", "128", "148"] for i, (m, pr, t, rd, wr) in enumerate(
        [(1, 0, "100", "1000", "0.5"), (4, 1, "200", "400", "0.4"), (4, 1, "210", "400", "0.4"), (4, 1, "205", "400", "0.4"),
         (4, 1, "20", "10", "0.01")])]
    raw = tmp_path / "raw.csv"
    with open(raw, "w", newline="") as fh:
        import csv
        w = csv.writer(fh, quoting=csv.QUOTE_ALL)
        w.writerow(hdr); w.writerow(units)
        for r in rows:
            w.writerow(r)
    ncu_summary.main(["step", str(raw), "--workload", "w", "--tag", "t", "--command", "ncu ...", "--out-dir", str(tmp_path)])
    md = (tmp_path / "t_step_w.md").read_text()
    assert "tc_gemm_kernel<1, 0, 0> TC_FWD_SWIGLU" in md and "| 100.0 | 1000.0 | 500.0 |" in md
    tr = json.loads((tmp_path / "traffic.json").read_text())["w"]["stages"]
    assert abs(tr["gemm1_swiglu"] - 1.5e9) < 1 and abs(tr["wgrad"] - 0.8e9) < 1
    lc = tmp_path / "l.csv"
    with open(lc, "w", newline="") as fh:
        w = csv.writer(fh, quoting=csv.QUOTE_ALL)
        w.writerow(["ID", "Kernel Name", "Metric Name", "Metric Unit", "Metric Value"])
        w.writerow(["0", k % (0, 0), "gpu__time_duration.sum", "ns", "2000"])
        w.writerow(["1", k % (0, 0), "gpu__time_duration.sum", "ns", "4000"])
    ncu_summary.main(["launches", str(lc), "--workload", "w", "--tag", "t", "--command", "ncu ...", "--out-dir", str(tmp_path)])
    assert "| `tc_gemm_kernel<0, 0, 0> TC_FWD` | 2 | 3.0 | 100.0% |" in (tmp_path / "t_launches_w.md").read_text()
