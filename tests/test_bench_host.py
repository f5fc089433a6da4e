"""Host-side logic of bench.py on CPU: the reference arm under torchrun (world size 2, rank 0 alone prints), the
max-over-ranks reduction over gloo, and the roofline bookkeeping.  No GPU, no CUDA library calls."""
import json
import os
import socket
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r measured (1 + r) s for the step and (0.5 - 0.1 r) s for the kernel: the job is as slow as its slowest rank
    t_all, t_sim = bench.max_over_ranks([1.0 + rank, 0.5 - 0.1 * rank])
    out[rank] = (t_all, t_sim, bench.whole_job_value(100.0, 3, world, t_all))
    dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    port = _free_port()
    with mp.Manager() as man:
        out = man.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        res = dict(out)
    for r in (0, 1):
        t_all, t_sim, val = res[r]
        assert t_all == 2.0 and t_sim == 0.5
        assert val == pytest.approx(2 * 100.0 * 3 / 2.0)


def test_max_over_ranks_single_process():
    assert bench.max_over_ranks([0.25, 4.0]) == [0.25, 4.0]


def test_reference_arm_under_torchrun_world2():
    """rank 0 alone runs the oracle and prints ONE JSON line; the other rank exits 0 without work"""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0", "--workload", "T3", "--ref-budget", "2e7"]
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"] > 0
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["vs_baseline"] is None and d["higher_is_better"] is True


def test_roofline_bookkeeping():
    """T_roof = max(bytes / HBM, MUFU ops / rate, FP32 instructions / rate); frac = T_roof / t"""
    sg = {"steps": 1000, "active_updates": 33000 * 9, "is3d": True}
    nt, hbm, mhz = 9, 6544.0, 1965.0
    r = bench.roofline(sg, nt, 1e-3, hbm, mhz, "measured")
    u = 33000 * nt
    t_hbm = 1000 * (8 + 16 + 24 * nt) / (hbm * 1e9)
    t_mufu = u * (1 + 1 / nt) / (148 * 16 * mhz * 1e6)
    t_fp32 = u * (8 + 4 / nt) / (148 * 128 * mhz * 1e6)
    assert r["frac"] == pytest.approx(max(t_hbm, t_mufu, t_fp32) / 1e-3)
    assert r["bound"] in ("hbm", "alu") and r["frac"] == pytest.approx(r["achieved"] / r["peak"])
    assert r["hbm_frac"] == pytest.approx(t_hbm / 1e-3) and r["mufu_frac"] == pytest.approx(t_mufu / 1e-3)


def test_own_arm_fails_loudly_without_gpu():
    if torch.cuda.is_available():
        pytest.skip("needs a box without CUDA")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--workload", "T3"], capture_output=True, text=True, cwd=ROOT)
    assert p.returncode != 0 and "no CUDA device" in (p.stderr + p.stdout)
