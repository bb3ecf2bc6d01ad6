#!/usr/bin/env python
"""bench.py — one SPD cycle ("step") of the 9B-class config on B200, through the C ABI.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 9b_n4] [--impl reference]

A step is one pass of the whole hot path (PDM, L/n stage-batched layer passes, verify,
accept/rollback) over one batch-1 sequence of synthetic inputs (seeded bf16 N(0,0.02) weights, uniform
random prompt of the config's length, forced acceptance p = 1 so every timed step is the saturated
step: all n stages occupied, exit + verify).  Prints ONE JSON line (rank 0).

value      SPD step latency in us with everything resident in HBM: K cycles enqueued back to back
           (spd_step_many), CUDA events on the library's stream, max over ranks.
e2e        the same latency through spd_step(): one host call per cycle, result struct copied
           device->host and the stream synchronised inside the timed region (host wall clock).
roofline   the fused cycle kernel (the only kernel of a step): algorithmic bytes of a saturated cycle
           (all layer weights + touched KV + tied matrix E once + W_p) / mean launch duration, against the
           measured copy bandwidth in MEASURED_PEAKS.json.
cpu_baseline  the oracle (oracle/, as it stands) timed on this box's host cores on a bounded sample.
--impl reference  times the oracle instead (the reference arm of this tier).
N > 1: the path is "replicas only": every rank runs an independent sequence; no collective
on the data path; value = max over ranks of the step latency, tokens/s and GB/s are summed.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import spd_inputs as si  # noqa: E402

METRIC = "SPD step latency (us), batch-1 tokens/s, achieved HBM GB/s vs ~8 TB/s"
NOMINAL_HBM_GBS = 8000.0
FALLBACK_HBM_GBS = 6650.0   # /opt/skills/guides/B200_PROFILING.md fallback


# ------------------------------------------------------------------------------------ helpers
def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_ read+write)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md, 6.65 TB/s)"


def recorded_traffic(kernel: str):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full capture
    (profiles/traffic.csv; the command that made it is in the .md named in its `source` column), or None."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        for line in open(p).read().splitlines()[1:]:
            name, nbytes = line.split(",")[:2]
            if name == kernel:
                return int(nbytes)
    except Exception:
        return None
    return None


class ClockSampler:
    """Samples SM clock and throttle reasons DURING the timed region (pynvml, ~10 ms period)."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting"}

    def __init__(self, device: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            visible = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = device
            if visible:
                try:
                    idx = int(visible.split(",")[device])
                except Exception:
                    idx = device
            self.h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        while not self._stop.is_set():
            try:
                self.samples.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                mask = self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for bit, name in self.REASONS.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.01)

    def start(self):
        if self.nv:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr:
            self._stop.set()
            self._thr.join()
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def aggregate(local: dict, world: int) -> dict:
    """Max over ranks for times, sum for rates (replicas).  torch.distributed must be initialised if world > 1."""
    if world == 1:
        return dict(local)
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    out = dict(local)
    for key, op in (("step_us", dist.ReduceOp.MAX), ("e2e_us", dist.ReduceOp.MAX), ("kernel_us", dist.ReduceOp.MAX),
                    ("tokens_per_s", dist.ReduceOp.SUM), ("hbm_gbs", dist.ReduceOp.SUM), ("gpu_launches", dist.ReduceOp.SUM)):
        if local.get(key) is None:
            continue
        t = torch.tensor([float(local[key])], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=op)
        out[key] = float(t.item())
    return out


# ------------------------------------------------------------------------------------ oracle legs
def oracle_saturated_cycle_us(shape, weights_np, context: int, samples: int, budget_s: float = 150.0):
    """Times the oracle's saturated cycle (fill n: all stages + PDM + exit/verify).  KV cache = seeded
    filler rows (values do not change the time); drafts are the PDM's own, so after every reject the
    pipeline refills and every n-th cycle is saturated.  Returns (median us, cycles timed, threads)."""
    from oracle import Oracle, num_threads
    n = shape.n_stages
    ora = Oracle(shape, weights_np, max_seq=context + (samples + 2) * (n + 1) + 16)
    for l in range(shape.n_layers):
        k, v = si.make_kv_filler(shape, l, context)
        ora.load_kv(l, k, v)
    ora.assume_prefilled(context, 1)
    times, t_start = [], time.time()
    while len(times) < samples:
        fill = ora.fill
        t0 = time.perf_counter()
        r = ora.step()
        dt = time.perf_counter() - t0
        if fill == n and r.exited:
            times.append(dt * 1e6)
        if time.time() - t_start > budget_s and times:
            break
    ora.close()
    return statistics.median(times), len(times), num_threads()


def run_reference(args, shape):
    """--impl reference: the oracle as it stands, on this box's host cores (rank 0 only)."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    t0 = time.time()
    w = si.make_weights(shape, seed=args.seed)
    ctx_len = shape.prompt_len + shape.gen_len // 2
    # bounded sample: each timed "step" is one saturated oracle cycle; at most ~150 s in total
    probe, _, threads = oracle_saturated_cycle_us(shape, w, ctx_len, 1)
    k = max(1, min(args.steps, int(150e6 / probe)))
    med, timed, threads = oracle_saturated_cycle_us(shape, w, ctx_len, k)
    a = 1.0
    full = step_bytes(shape, ctx_len)["full"]
    line = {"impl": "reference", "metric": METRIC, "value": med, "unit": "us", "n_gpus": 0, "steps": args.steps,
            "steps_timed": timed, "warmup": args.warmup, "ms_per_step": med / 1e3, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32 tensors, f64 accumulation (oracle)", "data": "synthetic",
            "config": {"workload": f"{shape.name}: saturated SPD cycle, context {ctx_len}", "forced_p": 1.0},
            "tokens_per_s": a * 1e6 / med, "hbm_gbs": full / med / 1e3,
            "cpu_baseline": {"value": med, "unit": "us", "cores": threads, "kind": "oracle",
                             "sample": f"{timed} saturated cycles (fill {shape.n_stages}) of {shape.name}; KV cache = "
                                       f"seeded filler rows of length {ctx_len}; each requested step is one such cycle, "
                                       f"count bounded to ~150 s"},
            "e2e": {"value": med, "unit": "us", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "wall_s": time.time() - t0}
    print(json.dumps(line), flush=True)


def step_bytes(shape, context_len, fill=None, exited=True, pdm=True):
    from paper_2605_30852_b200 import reporting
    return reporting.step_bytes(shape, context_len, fill, exited, pdm)


# ------------------------------------------------------------------------------------ GPU arm
def run_gpu(args, shape):
    import torch
    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the SPD path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    import paper_2605_30852_b200 as spd

    n, P, G = shape.n_stages, shape.prompt_len, shape.gen_len
    need = max(G, 2 * args.steps + args.warmup + 4 * n) + n + 8
    max_seq = P + need + 2 * n + 640          # head-room for the chunked step_many calls
    t_setup = time.time()
    w_np = si.make_weights(shape, seed=args.seed + rank)        # every replica its own sequence
    w_dev = spd.upload_weights(w_np, local_rank)
    eng = spd.SPD(shape, w_dev, max_seq=max_seq, device=local_rank)
    if args.engine is not None:
        eng.set_option(spd.OPT.ENGINE, args.engine)
    if args.chains is not None:
        eng.set_option(spd.OPT.CHAINS, args.chains)
    prompt = si.make_prompt(shape, args.seed + rank)
    first = eng.prefill(prompt)
    # the step before the path (untimed in the paper): the batched tensor-core prefill, timed once warm
    pe0, pe1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    pe0.record(eng.stream_main)
    first2 = eng.prefill(prompt)
    pe1.record(eng.stream_main)
    torch.cuda.synchronize()
    assert first2 == first
    prefill_ms = pe0.elapsed_time(pe1)
    # truth table = the library's own greedy tokens (C-2.20): unforced SPD is lossless, so its emitted
    # tokens are the greedy continuation; then rewind to the prefill state.
    toks, _ = eng.generate(need, chunk=64)
    truth = np.array([first] + toks, dtype=np.int32)[:need]
    t_setup = time.time() - t_setup

    def rewind(p):
        eng.rollback(P, first)
        eng.set_forced(truth, p, args.seed)

    # ---- headline: saturated cycles at p = 1 ------------------------------------------------
    rewind(1.0)
    eng.step_many(n)                                            # fill the pipeline (untimed)
    done = 0
    while done < args.warmup:
        m = min(512, args.warmup - done)
        eng.step_many(m)
        done += m
    stream = eng.stream_main
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    clocks = ClockSampler(local_rank)
    _, _, l0 = eng.counters()
    if world > 1:
        torch.distributed.barrier()
    torch.cuda.synchronize()
    clocks.start()
    ev0.record(stream)
    res, done = [], 0
    while done < args.steps:
        m = min(512, args.steps - done)
        res += eng.step_many(m)
        done += m
    ev1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        torch.distributed.barrier()
    clk = clocks.stop()
    step_us = ev0.elapsed_time(ev1) * 1e3 / args.steps
    _, _, l1 = eng.counters()
    launches = l1 - l0
    assert all(r.fill == n and r.exited and r.accepted for r in res), "timed steps must be saturated accept steps"
    timed_lat = [us for _, us in cycle_latencies_us(eng, res, 512)]      # device stamps of the timed cycles themselves
    ctx_mid = (res[0].committed_len + res[-1].committed_len) // 2 + n // 2
    by = step_bytes(shape, ctx_mid)

    phases = None
    if args.phase_profile:     # per-phase stamps of saturated cycles (the pipeline is still saturated at p = 1)
        phases = phase_table(eng, shape)

    # ---- e2e: one host call per cycle, result D2H + sync inside the timed region -----------------
    ke = min(args.steps, max(50, args.steps // 4))
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(ke):
        eng.step()
    e2e_us = (time.perf_counter() - t0) * 1e6 / ke
    d2h = 36 + eng_state_bytes()

    # ---- acceptance sweep (tokens/s at the config's p values; not part of the timed K steps) --------
    sweep = {}
    fill_samples = []
    SW_CHUNK = 32
    for p in shape.p_sweep:
        rewind(p)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        toks_p, log, unread = [], [], 0
        while len(toks_p) < G - 1:
            chunk_log = eng.step_many(SW_CHUNK)
            log += chunk_log
            toks_p += [r.emitted_token for r in chunk_log if r.exited]
            unread += SW_CHUNK
            if unread + SW_CHUNK > 1024:                      # the device keeps the stamps of the last 1024 cycles
                fill_samples += cycle_latencies_us(eng, log[-unread:], SW_CHUNK)
                unread = 0
        e1.record(stream)
        torch.cuda.synchronize()
        if unread:
            fill_samples += cycle_latencies_us(eng, log[-unread:], SW_CHUNK)
        ms = e0.elapsed_time(e1)
        emitted = sum(r.exited for r in log)
        ok = ([first] + toks_p)[:G] == list(truth[:G])
        sweep[str(p)] = {"steps": len(log), "alpha": emitted / len(log), "tokens_per_s": emitted / ms * 1e3,
                         "mean_step_us": ms * 1e3 / len(log), "lossless_vs_greedy": bool(ok),
                         "fill_hist": {str(a): sum(1 for r in log if r.fill == a) for a in range(1, n + 1)}}

    # ---- sampling verification (NEXT-2; PAPER.md:141 T=1, top-k 50): cycle latency next to the greedy path on the
    # same fill pattern.  Random-init PDM and target supports are disjoint, so both runs reject at every exit
    # (fill 1..n round robin); the difference is the cost of keeping the logit vectors + the top-k selection.
    def timed_cycles(k):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        eng.step_many(n)
        e0.record(stream)
        log = eng.step_many(k)
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e3 / k, log

    ks = min(256, need - 2 * n)
    rewind(-1.0)                                                # greedy, the PDM's own drafts
    g_us, g_log = timed_cycles(ks)
    eng.rollback(P, first)
    eng.set_sampling(1.0, 50, args.seed)
    s_us, s_log = timed_cycles(ks)
    eng.set_sampling(1.0, 0, 0)
    hist = lambda log: {str(a): sum(1 for r in log if r.fill == a) for a in range(1, n + 1)}
    sampling = {"temperature": 1.0, "top_k": 50, "cycles": ks, "mean_step_us": s_us, "greedy_same_drafts_mean_step_us": g_us,
                "overhead_us": s_us - g_us, "accept_rate": sum(r.accepted for r in s_log) / max(1, sum(r.exited for r in s_log)),
                "fill_hist": hist(s_log), "greedy_fill_hist": hist(g_log)}

    # ---- ... and at SATURATION.  Random-init drafts are never accepted under sampling, so the saturated sampling cycle
    # (fill n, exit, target top-k, accept test) is timed on an "echo" re-initialisation of the SAME device tensors:
    # W_o = W_down = 0 (every layer leaves the residual stream untouched; all bytes are still streamed) and
    # W_p = [I 0 .. 0], so the PDM's logits for a token equal the target's bit for bit, Q = P, and every draft is
    # accepted (u * Q(x) < P(x) for every u < 1).  The greedy cycle is timed on the same tensors beside it.
    eng.close()

    # ---- NEXT-1: the paper's Pipeline Draft Module (PAPER.md:71, :91-100, :121 "L_s ~ L/n - 1", :139, :299) in place of the
    # simplified one: L_s = L/n - 1 layers (>= 1), a 32000-entry head; saturated cycles at forced p = 1 on the same target.
    paper = None
    if not args.no_paper_pdm:
        Ls, Vs = max(1, shape.n_layers // n - 1), min(32000, shape.vocab)
        pw = si.make_pdm_weights(shape, Ls, Vs, seed=args.seed + rank)
        eng2 = spd.SPD(shape, w_dev, max_seq=P + 4 * args.steps + 8 * n + 64, device=local_rank)
        eng2.attach_pdm(spd.upload_pdm_weights(pw, local_rank))
        if args.engine is not None:
            eng2.set_option(spd.OPT.ENGINE, args.engine)
        if args.chains is not None:
            eng2.set_option(spd.OPT.CHAINS, args.chains)
        s2 = eng2.stream_main
        q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        eng2.prefill(prompt)
        q0.record(s2)
        f2 = eng2.prefill(prompt)
        q1.record(s2)
        torch.cuda.synchronize()
        pdm_prefill_ms = q0.elapsed_time(q1)
        eng2.set_forced(truth, 1.0, args.seed)
        eng2.step_many(n + args.warmup)
        kp = min(args.steps, 200)
        q0.record(s2)
        plog = eng2.step_many(kp)
        q1.record(s2)
        torch.cuda.synchronize()
        pdm_cycle_us = q0.elapsed_time(q1) * 1e3 / kp
        m_anch = si.pdm_anchor_count(shape.n_layers)
        d = shape.d_model
        Lt, anchors = shape.n_layers, sorted({0, shape.n_layers // 4, shape.n_layers // 2, 3 * shape.n_layers // 4, shape.n_layers - 1})
        # a saturated draft has one row per depth k = 0 .. n; row k reads FC_f(k), (f(k) + 1) d x d (Eq. 3-4)
        fc_bytes = sum(2 * d * d * sum(1 for b in anchors if b <= min(Lt, k * (Lt // n))) for k in range(n + 1))
        pdm_bytes = fc_bytes + 2 * Ls * shape.layer_params() + 2 * Vs * d + (n + 1) * Ls * 4 * shape.n_kv_heads * shape.head_dim * ctx_mid
        paper = {"pdm_layers": Ls, "pdm_vocab": Vs, "rows_per_draft": n + 1, "cycles": kp,
                 "cycle_us_with_paper_pdm": pdm_cycle_us, "cycle_us_simplified_pdm": step_us, "pdm_cost_us": pdm_cycle_us - step_us,
                 "pdm_algorithmic_bytes": pdm_bytes, "pdm_gbs": pdm_bytes / max(pdm_cycle_us - step_us, 1e-9) / 1e3,
                 "masked_on_a_dedicated_gpu": bool(pdm_cycle_us - step_us < step_us),
                 "note": "the draft's kernels run in front of the cycle kernel on the same GPU (the paper hides them on a dedicated rank, "
                         "PAPER.md:119); 'masked' = the draft takes less than one cycle (PAPER.md:121)",
                 "prefill_ms_incl_pdm_rows": pdm_prefill_ms, "all_saturated_accepts": all(r.fill == n and r.accepted for r in plog),
                 "first_token_matches": bool(f2 == first)}
        eng2.close()
        del eng2, pw

    for l in range(shape.n_layers):
        w_dev["wo"][l].zero_()
        w_dev["w_down"][l].zero_()
    w_dev["pdm_proj"].zero_()
    w_dev["pdm_proj"][:, :shape.d_model].fill_diagonal_(0x3F80)          # bf16 1.0
    w_dev["pdm_norm"].copy_(w_dev["final_norm"])
    eng = spd.SPD(shape, w_dev, max_seq=P + 2 * ks + 8 * n + 64, device=local_rank)
    if args.engine is not None:
        eng.set_option(spd.OPT.ENGINE, args.engine)
    if args.chains is not None:
        eng.set_option(spd.OPT.CHAINS, args.chains)
    stream = eng.stream_main
    eng.set_sampling(1.0, 50, args.seed)
    first_e = eng.prefill(prompt)
    ss_us, ss_log = timed_cycles(ks)
    eng.set_sampling(1.0, 0, 0)
    eng.rollback(P, first_e)
    sg_us, sg_log = timed_cycles(ks)
    acc = lambda log: sum(r.accepted for r in log) / max(1, sum(r.exited for r in log))
    sampling["saturated"] = {"init": "echo (W_o = W_down = 0, W_p = [I 0 .. 0]): Q = P, every draft is accepted",
                             "cycles": ks, "mean_step_us": ss_us, "greedy_mean_step_us": sg_us, "overhead_us": ss_us - sg_us,
                             "accept_rate": acc(ss_log), "greedy_accept_rate": acc(sg_log),
                             "tokens_per_s": sum(r.exited for r in ss_log) / (ss_us * ks) * 1e6,
                             "all_fill_n": all(r.fill == n for r in ss_log) and all(r.fill == n for r in sg_log)}

    local = {"step_us": step_us, "e2e_us": e2e_us, "kernel_us": step_us, "tokens_per_s": 1e6 / step_us,
             "hbm_gbs": by["full"] / step_us / 1e3, "gpu_launches": launches}
    tot = aggregate(local, world)
    if rank != 0:
        eng.close()
        return
    peak, peak_src = measured_peak()
    achieved = by["full"] / tot["kernel_us"] / 1e3               # GB/s per GPU
    kname = {1: "k_spd_cycle", 2: "k_spd_cycle2"}.get(eng.get_option(spd.OPT.ENGINE), "reference engine (kernel per op)")
    line = {
        "metric": METRIC, "value": tot["step_us"], "unit": "us", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": tot["step_us"] / 1e3, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16 weights, f32 activations/accumulation", "data": "synthetic",
        "config": {"workload": f"{shape.name}: d={shape.d_model} L={shape.n_layers} n={n} F={shape.d_ffn} V={shape.vocab}, "
                               f"prompt {P}, saturated cycles at forced p=1.0 (context ~{ctx_mid})",
                   "engine": ENGINE_NAMES[eng.get_option(spd.OPT.ENGINE)], "chains": eng.get_option(spd.OPT.CHAINS),
                   "l2": "working set %.1f GB per step >> 126 MB L2: no flush needed" % (by["full"] / 1e9),
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "tokens_per_s": tot["tokens_per_s"], "hbm_gbs": tot["hbm_gbs"],
        "frac_of_8tbs": {"strict": by["strict"] / tot["kernel_us"] / 1e3 / NOMINAL_HBM_GBS,
                         "full": by["full"] / tot["kernel_us"] / 1e3 / NOMINAL_HBM_GBS},
        "roofline": {"bound": "hbm", "kernel": kname, "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "peak_source": peak_src,
                     "frac_note": "the peak is a torch copy_ (read + write); a read-only stream can exceed it (frac > 1 is not an "
                                  "error) - frac_of_8tbs.strict is the north_star fraction", "algorithmic_bytes": by["full"],
                     "algorithmic_bytes_strict": by["strict"], "launch_us": tot["kernel_us"],
                     "traffic": recorded_traffic(kname)},
        "e2e": {"value": tot["e2e_us"], "unit": "us", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": d2h,
                "note": "spd_step(): launch + result/state D2H + stream sync per cycle; the cycle has no per-step host input "
                        "(ring, KV and lengths live on the device)"},
        "step_us_stats": {**percentiles(timed_lat), "unit": "us",
                          "source": "finish-stamp differences (%globaltimer, SPD_DBG_CYCLE_TIMES) of the timed back-to-back cycles"},
        "by_fill": by_fill_table(shape, fill_samples, peak),
        "prefill": prefill_report(shape, P, prefill_ms), "paper_pdm": paper, "phase_profile": phases,
        "gpu_launches": int(tot["gpu_launches"]), "clocks": clk, "p_sweep": sweep, "sampling": sampling,
        "setup_s": t_setup,
    }
    if world == 1 and not args.no_cpu_baseline:
        med, timed, threads = oracle_saturated_cycle_us(shape, w_np, ctx_mid, 3, budget_s=60.0)
        line["cpu_baseline"] = {"value": med, "unit": "us", "cores": threads, "kind": "oracle",
                                "sample": f"{timed} saturated cycles (fill {n}) of {shape.name}, KV cache = seeded filler rows "
                                          f"of length {ctx_mid}"}
    print(json.dumps(line), flush=True)
    eng.close()


ENGINE_NAMES = {0: "reference (kernel per op)", 1: "fused persistent cycle kernel k_spd_cycle (one stage chain per CTA)",
                2: "fused persistent cycle kernel k_spd_cycle2 (multiplexed stage chains)"}
PHASE_NAMES = {0: "PDM", 1: "QKV", 2: "ATTN", 3: "O", 4: "GATEUP", 5: "DOWN", 6: "HEAD"}


def phase_table(eng, shape, cycles: int = 8) -> dict:
    """Per-phase breakdown of the fused cycle kernel from its own clock stamps (SPD_OPT_PHASE_PROFILE; not under a
    profiler): mean over CTAs and over `cycles` saturated cycles of wait (this CTA's last tile of the previous phase ->
    its group's barrier open), stage (activation vector into shared memory, RMSNorm) and consume (streaming the phase's
    tiles), in us, per phase type; `per_cycle_us` = (wait + stage + consume) x occurrences."""
    import paper_2605_30852_b200 as spd
    per = shape.n_layers // shape.n_stages
    npz = 2 + 5 * per
    eng.set_option(spd.OPT.PHASE_PROFILE, 1)
    acc = {}
    two_chain = None
    for _ in range(cycles):
        eng.step()
        pr = eng.phase_profile().astype(np.int64)                 # [cta, phase, stamp]
        c0, g0, c1, g1 = pr[0, 167, 0], pr[0, 167, 1], pr[0, 167, 4], pr[0, 167, 5]
        mhz = (c1 - c0) / max(g1 - g0, 1) * 1e3                   # SM clocks per us
        nvis = int(np.count_nonzero(pr[0, :167, 2]))
        if nvis != npz:                                           # engine 2: stamps are filed per VISIT (phase x chain)
            two_chain = phase_table_two_chain(pr, per, mhz, two_chain)
            continue
        ncta = int(np.count_nonzero(pr[:, npz - 1, 2]))
        for p in range(npz):
            t = 0 if p == 0 else (6 if p == npz - 1 else 1 + (p - 1) % 5)
            s0, s1, s2 = pr[:ncta, p, 0], pr[:ncta, p, 1], pr[:ncta, p, 2]
            prev = pr[:ncta, p - 1, 2] if p > 0 else pr[:ncta, 167, 0]
            ok = (s0 > 0) & (s2 >= s1) & (s1 >= s0) & (prev > 0)
            if not ok.any():
                continue
            a = acc.setdefault(t, {"wait": [], "stage": [], "consume": []})
            a["wait"].append(float(np.mean((s0 - prev)[ok])) / mhz)
            a["stage"].append(float(np.mean((s1 - s0)[ok])) / mhz)
            a["consume"].append(float(np.mean((s2 - s1)[ok])) / mhz)
    eng.set_option(spd.OPT.PHASE_PROFILE, 0)
    if two_chain:
        return finish_two_chain(two_chain)
    out = {}
    for t, a in sorted(acc.items()):
        count = 1 if t in (0, 6) else per
        w, st, co = (float(np.mean(a[k])) for k in ("wait", "stage", "consume"))
        out[PHASE_NAMES[t]] = {"count": count, "wait_us": w, "stage_us": st, "consume_us": co, "per_cycle_us": (w + st + co) * count}
    return out


PHASE2_NAMES = ["QKV", "ATTN", "O", "GATEUP", "DOWN_A", "DOWN_B"]


def phase_table_two_chain(pr, per, mhz, acc):
    """Engine 2 (spd_mega2.cu): visit v of a CTA = PDM (0), then (phase, chain) pairs, then HEAD.  `wait` = end of the previous
    visit -> this visit's inputs handed over by the stager (dependency + staging, hidden when the stager is ahead),
    `consume` = streaming the visit's tiles.  Accumulates sums per (phase type, chain); returns the running table."""
    acc = acc or {"_n": 0}
    acc["_n"] += 1
    for cta in range(pr.shape[0]):
        nv = int(np.count_nonzero(pr[cta, :167, 2]))
        if nv < 2 or (nv - 2) % (6 * per):
            continue
        m = (nv - 2) // (6 * per)
        for v in range(nv):
            if v == 0:
                name = "PDM"
            elif v == nv - 1:
                name = "HEAD"
            else:
                pl, j = divmod(v - 1, m) if m else (0, 0)
                name = f"{PHASE2_NAMES[pl % 6]}.c{j}"
            s0, s1, s2 = pr[cta, v, 0], pr[cta, v, 1], pr[cta, v, 2]
            prev = pr[cta, v - 1, 2] if v > 0 else pr[cta, 167, 0]
            a = acc.setdefault(name, {"wait_us": 0.0, "stage_us": 0.0, "consume_us": 0.0, "visits": 0})
            a["wait_us"] += float(s0 - prev) / mhz
            a["stage_us"] += float(s1 - s0) / mhz
            a["consume_us"] += float(s2 - s1) / mhz
            a["visits"] += 1
    return acc


def finish_two_chain(acc, ncta=148):
    out = {}
    n = acc.pop("_n")
    for name, a in acc.items():
        k = a["visits"]
        out[name] = {"visits_per_cta_cycle": k / (n * ncta), "wait_us": a["wait_us"] / k, "stage_us": a["stage_us"] / k,
                     "consume_us": a["consume_us"] / k,
                     "per_cycle_us": (a["wait_us"] + a["stage_us"] + a["consume_us"]) / (n * ncta)}
    return out


def percentiles(x) -> dict:
    a = np.asarray(x, dtype=np.float64)
    if a.size == 0:
        return {"n": 0}
    return {"n": int(a.size), "median": float(np.median(a)), "p10": float(np.percentile(a, 10)),
            "p90": float(np.percentile(a, 90)), "mean": float(a.mean())}


def cycle_latencies_us(eng, log, chunk: int):
    """Per-cycle step latency from the device's own stamps (SPD_DBG_CYCLE_TIMES): the difference of the finish stamps
    (%globaltimer) of consecutive back-to-back cycles.  `log` = the StepResults of cycles enqueued in chunks of
    `chunk` (a host sync separates chunks, so the first cycle of a chunk has no back-to-back predecessor and is
    left out).  Only the last 1024 cycles are on the device.  Returns [(StepResult, latency_us)]."""
    tail = log[-1024:]
    off = len(log) - len(tail)
    ts = eng.cycle_times([r.step_index for r in tail])
    out = []
    for j in range(1, len(tail)):
        if (off + j) % chunk == 0 or tail[j].step_index != tail[j - 1].step_index + 1:
            continue
        out.append((tail[j], (ts[j, 1] - ts[j - 1, 1]) / 1e3))
    return out


def by_fill_table(shape, samples, peak_gbs: float) -> dict:
    """latency and GB/s per fill level a.  B(a) = (a/n) layer weights + KV rows of a tokens + E + W_p
    (reporting.step_bytes; a cycle without an exit still runs the PDM's pass over the tied E)."""
    n = shape.n_stages
    out = {}
    for a in range(1, n + 1):
        for exited in (0, 1):
            sel = [(r, us) for r, us in samples if r.fill == a and r.exited == exited]
            if not sel:
                continue
            st = percentiles([us for _, us in sel])
            ctx = int(np.median([r.committed_len for r, _ in sel])) + a // 2
            by = step_bytes(shape, ctx, fill=a, exited=bool(exited))
            gbs = by["full"] / st["median"] / 1e3
            out[f"{a}{'' if exited == (a == n) else ('+exit' if exited else '-noexit')}"] = {
                **st, "unit": "us", "exited": bool(exited), "algorithmic_bytes": by["full"], "algorithmic_bytes_strict": by["strict"],
                "gbs": gbs, "frac_of_8tbs": gbs / NOMINAL_HBM_GBS, "frac_of_8tbs_strict": by["strict"] / st["median"] / 1e3 / NOMINAL_HBM_GBS,
                "frac_of_measured_peak": gbs / peak_gbs}
    return out


def prefill_report(shape, P: int, ms: float) -> dict:
    """spd_prefill of the config's prompt (NEXT-4; outside the paper's timed region).  Useful flops = 2 x tokens x layer
    parameters (GEMMs only); the tensor cores execute 3x that (fp32 activations as three exact bf16 parts).  Peak = the
    measured dense bf16 rate in MEASURED_PEAKS.json (sustained), else the nominal 2250 TFLOP/s."""
    useful = 2.0 * P * shape.layer_params() * shape.n_layers
    peak, src = 2250.0, "nominal (B200 dense bf16)"
    try:
        mp = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        peak, src = float(mp.get("bf16_tflops_sustained", mp["bf16_tflops"])), "measured (MEASURED_PEAKS.json, torch.matmul bf16 sustained)"
    except Exception:
        pass
    t = ms / 1e3
    return {"tokens": P, "ms": ms, "tokens_per_s": P / t, "useful_tflops": useful / t / 1e12, "mma_tflops": 3.0 * useful / t / 1e12,
            "bound": "tensor", "peak_tflops": peak, "peak_source": src, "frac_mma": 3.0 * useful / t / 1e12 / peak,
            "note": "whole call (GEMMs + attention + elementwise kernels + the final head cycle), CUDA events, warm"}


def eng_state_bytes() -> int:
    return 608   # sizeof(StepState): the state mirror copied to the host by every spd_step (csrc/spd_dev.cuh)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=400)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", default="9b_n4", choices=sorted(si.CONFIGS))
    ap.add_argument("--impl", default="spd", choices=["spd", "reference"])
    ap.add_argument("--engine", type=int, default=None, help="0 reference engine, 1 / 2 fused engines (default: library default = 2)")
    ap.add_argument("--chains", type=int, default=None, help="engine 2: stage chains per CTA, 1..4 (default: library default)")
    ap.add_argument("--seed", type=int, default=1234)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--phase-profile", action="store_true", help="add the fused kernel's per-phase breakdown (its own clock stamps)")
    ap.add_argument("--no-paper-pdm", action="store_true", help="skip the NEXT-1 leg (the paper's PDM in place of the simplified one)")
    args = ap.parse_args()
    shape = si.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, shape)
    else:
        run_gpu(args, shape)


if __name__ == "__main__":
    main()
