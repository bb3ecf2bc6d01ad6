"""GPU-vs-oracle parity harness (used by the -m gpu tests and __graft_entry__.smoke()).

Runs the CUDA library and the CPU oracle on the same seeded inputs, cycle by cycle, and compares:
step results (token ids, accept bits, fill, committed length: exact), per-depth hidden states, PDM
pre-norm vector, logits, KV lengths (exact) and KV rows.  Token mismatches are classified with the
oracle's top-1/top-2 margin: below TAU * max|logit| it is a near-tie (fp32
re-association can legitimately flip it) and the caller retries with the next seed; above, a failure.
"""
from __future__ import annotations

import dataclasses

import numpy as np

import spd_inputs as si
from oracle import Oracle

TAU = 1e-4          # near-tie threshold on (top1 - top2) / max|logit|
CONTRACT = 2e-2     # north_star: hidden states and logits within max relative error 2e-2


def rel_err(a, b) -> float:
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    den = float(np.max(np.abs(b)))
    return float(np.max(np.abs(a - b)) / (den if den > 0 else 1.0))


@dataclasses.dataclass
class Report:
    status: str = "ok"            # "ok" | "near_tie" | "fail"
    detail: str = ""
    steps: int = 0
    emitted: int = 0
    max_hidden_err: float = 0.0
    max_logit_err: float = 0.0
    max_pdm_err: float = 0.0
    kv_flip_frac: float = 0.0
    min_margin: float = 1.0
    accepts: int = 0
    rejects: int = 0
    tokens: list = dataclasses.field(default_factory=list)


def kv_compare(gpu, ora, layers, rows, rep: Report, tol: float):
    """bf16 K/V rows: every entry within one bf16 ulp of the oracle's plus fp slack; report flip fraction."""
    for l in layers:
        for which in (0, 1):
            g = si.bf16_bits_to_f32(gpu.kv(l, which, rows)).astype(np.float64)
            o = si.bf16_bits_to_f32(ora.kv(l, which, rows)).astype(np.float64)
            bad = g != o
            rep.kv_flip_frac = max(rep.kv_flip_frac, float(bad.mean()) if bad.size else 0.0)
            lim = 2.0 ** -7 * np.abs(o) + tol * (np.max(np.abs(o)) if o.size else 0.0)
            if not np.all(np.abs(g - o) <= lim):
                rep.status, rep.detail = "fail", f"KV rows differ beyond one bf16 ulp (layer {l}, {'KV'[which]})"
                return False
    return True


def run_parity(shape, weights_np, dev_weights, prompt, n_tokens, forced=None, engine=None, tensor_every=1,
               tensor_tol=CONTRACT, check_logits=True, prefill_block=16, max_seq=None, spd_cls=None, gpu=None) -> Report:
    """forced = (truth tokens, p, seed) or None (the PDM's own drafts)."""
    from paper_2605_30852_b200 import SPD, OPT
    rep = Report()
    n = shape.n_stages
    ms = max_seq or (len(prompt) + n_tokens * (n + 1) + 2 * n + 8)
    ora = Oracle(shape, weights_np, max_seq=ms)
    own = gpu is None
    if own:
        gpu = (spd_cls or SPD)(shape, dev_weights, max_seq=ms)
    try:
        if engine is not None:
            gpu.set_option(OPT.ENGINE, engine)
        gpu.set_option(OPT.DEBUG_LOGITS, 1 if check_logits else 0)
        fo = ora.prefill(prompt, block=prefill_block)
        fg = gpu.prefill(prompt)
        gap, mx = ora.margin(0)
        rep.min_margin = gap / mx
        if fo != fg:
            if gap < TAU * mx:
                rep.status, rep.detail = "near_tie", "first token"
            else:
                rep.status, rep.detail = "fail", f"first token {fg} != oracle {fo} (margin {gap / mx:.2e})"
            return rep
        rep.tokens.append(fg)
        P = len(prompt)
        e = rel_err(gpu.hfin(P - 1), ora.hfin(P - 1))
        rep.max_hidden_err = max(rep.max_hidden_err, e)
        if e > tensor_tol:
            rep.status, rep.detail = "fail", f"prefill final hidden state rel err {e:.3e}"
            return rep
        if not np.array_equal(gpu.kv_len(), ora.kv_len()):
            rep.status, rep.detail = "fail", "KV lengths differ after prefill"
            return rep
        if not kv_compare(gpu, ora, sorted({0, shape.n_layers // 2, shape.n_layers - 1}), P, rep, tensor_tol):
            return rep
        if forced is not None:
            truth, p, seed = forced
            ora.set_forced(truth, p, seed)
            gpu.set_forced(truth, p, seed)
        while ora.emitted < n_tokens:
            ro = ora.step()
            rg = gpu.step()
            rep.steps += 1
            if tuple(ro) != tuple(rg):
                which = 0 if ro.emitted_token != rg.emitted_token else 1
                gap, mx = ora.margin(which)
                only_token = (ro._replace(emitted_token=0, draft_token=0, accepted=0, discarded=0, committed_len=0) ==
                              rg._replace(emitted_token=0, draft_token=0, accepted=0, discarded=0, committed_len=0))
                if only_token and gap < TAU * mx:
                    rep.status, rep.detail = "near_tie", f"step {rep.steps}: {'verify' if which == 0 else 'PDM'} margin {gap / mx:.2e}"
                else:
                    rep.status, rep.detail = "fail", f"step {rep.steps}: gpu {tuple(rg)} != oracle {tuple(ro)} (margin {gap / mx:.2e})"
                return rep
            if ro.exited:
                rep.emitted += 1
                rep.tokens.append(ro.emitted_token)
                rep.accepts += ro.accepted
                rep.rejects += 1 - ro.accepted
                g, m = ora.margin(0)
                rep.min_margin = min(rep.min_margin, g / m)
            g, m = ora.margin(1)
            rep.min_margin = min(rep.min_margin, g / m)
            if rep.steps % tensor_every == 0:
                fill, c, slots = gpu.ring()
                if fill != ora.fill or c != ora.committed_len:
                    rep.status, rep.detail = "fail", f"step {rep.steps}: ring fill/committed differ"
                    return rep
                for i in range(ora.fill):
                    pos, tok, k, h = ora.ring(i)
                    if slots[k] != (1, pos, tok):
                        rep.status, rep.detail = "fail", f"step {rep.steps}: depth {k} holds {slots[k]}, oracle ({pos},{tok})"
                        return rep
                    e = rel_err(gpu.hidden(k), h)
                    rep.max_hidden_err = max(rep.max_hidden_err, e)
                e = rel_err(gpu.last("pdm_prenorm"), ora.last("pdm_prenorm"))
                rep.max_pdm_err = max(rep.max_pdm_err, e)
                if check_logits:
                    e = rel_err(gpu.last("pdm_logits"), ora.last("pdm_logits"))
                    if ro.exited:
                        e = max(e, rel_err(gpu.last("exit_logits"), ora.last("exit_logits")))
                    rep.max_logit_err = max(rep.max_logit_err, e)
                if not np.array_equal(gpu.kv_len(), ora.kv_len()):
                    rep.status, rep.detail = "fail", f"step {rep.steps}: KV lengths differ"
                    return rep
                worst = max(rep.max_hidden_err, rep.max_pdm_err, rep.max_logit_err)
                if worst > tensor_tol:
                    rep.status, rep.detail = "fail", f"step {rep.steps}: tensor rel err {worst:.3e} > {tensor_tol}"
                    return rep
        c = ora.committed_len
        kv_compare(gpu, ora, sorted({0, shape.n_layers - 1}), c, rep, tensor_tol)
        return rep
    finally:
        ora.close()
        if own:
            gpu.close()


def run_parity_retry(make_inputs, seeds, **kw) -> Report:
    """make_inputs(seed) -> dict of run_parity kwargs.  Retries on near-ties with the next seed (C-4);
    returns the first clean report (its .detail lists the near-ties met on the way)."""
    notes = []
    for s in seeds:
        rep = run_parity(**make_inputs(s), **kw)
        if rep.status == "near_tie":
            notes.append(f"seed {s}: near-tie at {rep.detail}")
            continue
        rep.detail = "; ".join(notes + ([rep.detail] if rep.detail else []))
        return rep
    rep.detail = "; ".join(notes)
    return rep
