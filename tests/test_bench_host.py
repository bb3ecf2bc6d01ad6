"""Host-side logic of bench.py on CPU: the N > 1 reduction ("replicas only") over a
world-size-2 gloo group, the byte accounting of the roofline, and the argument/JSON contract pieces that
need no GPU."""
import json
import os
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import spd_inputs as si

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # rank r: a replica that is slower and moves fewer GB/s the higher its rank
        local = {"step_us": 2000.0 + 100.0 * rank, "e2e_us": 2100.0 + 50.0 * rank, "kernel_us": 1990.0 + 100.0 * rank,
                 "tokens_per_s": 500.0 - 10.0 * rank, "hbm_gbs": 5000.0 - 100.0 * rank, "gpu_launches": 7 + rank}
        q.put((rank, bench.aggregate(local, world)))
    finally:
        dist.destroy_process_group()


def _free_port():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.timeout(180)
def test_replica_aggregation_over_gloo_world_size_2():
    """Latencies: max over ranks; rates and launch counts: sum over ranks; every rank sees the same totals."""
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=150) for _ in procs)
    for p in procs:
        p.join(30)
        assert p.exitcode == 0
    for r in (0, 1):
        t = got[r]
        assert t["step_us"] == 2100.0 and t["e2e_us"] == 2150.0 and t["kernel_us"] == 2090.0
        assert t["tokens_per_s"] == 990.0 and t["hbm_gbs"] == 9900.0 and t["gpu_launches"] == 15.0


def test_aggregate_world_1_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    local = {"step_us": 1.0, "e2e_us": 2.0, "kernel_us": 3.0, "tokens_per_s": 4.0, "hbm_gbs": 5.0, "gpu_launches": 6}
    assert bench.aggregate(local, 1) == local


def test_step_bytes_by_fill_level():
    """B(a) = (a/n) W_layers + KV of a tokens + E + W_p; strict excludes E and W_p."""
    from paper_2605_30852_b200 import reporting as R
    s = si.CONFIGS["9b_n4"]
    T = 2176
    full = R.step_bytes(s, T)
    kv_row = 2 * s.n_kv_heads * s.head_dim * 2
    w_layers = s.layer_params() * 2 * s.n_layers
    assert full["strict"] == w_layers + kv_row * s.n_layers * T
    assert full["full"] - full["strict"] == s.vocab * s.d_model * 2 + s.n_stages * s.d_model * s.d_model * 2
    for a in range(1, s.n_stages + 1):
        b = R.step_bytes(s, T, fill=a, exited=(a == s.n_stages))
        assert b["strict"] == (w_layers + kv_row * s.n_layers * T) * a // s.n_stages
    # a cycle with neither a PDM nor an exit (prefill of a non-final prompt token) touches no head matrix
    b = R.step_bytes(s, T, fill=1, exited=False, pdm=False)
    assert b["full"] == b["strict"]


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_bench_gpu_arm_refuses_to_run_without_a_gpu():
    """The product arm has no CPU fallback: without a CUDA device bench.py exits non-zero and says why."""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--warmup", "1"],
                       capture_output=True, text=True, timeout=170)
    assert r.returncode != 0
    assert "no CUDA device" in (r.stderr + r.stdout)


@pytest.mark.timeout(280)
def test_reference_arm_prints_the_contract_line_on_the_tiny_config():
    """--impl reference times the oracle on the host cores and prints ONE JSON line with the base keys."""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "tiny",
                        "--steps", "3", "--warmup", "1"], capture_output=True, text=True, timeout=270)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["unit"] == "us" and j["higher_is_better"] is False
    assert j["cpu_baseline"]["kind"] == "oracle" and j["cpu_baseline"]["cores"] >= 1
    assert j["e2e"] == {"value": j["value"], "unit": "us", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert j["value"] > 0 and j["vs_baseline"] is None
