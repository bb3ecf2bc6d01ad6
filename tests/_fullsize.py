"""The full-size oracle tier: the CUDA path at BASELINE.json's full prompt lengths against what the
ORACLE computed there — the prefill result, the first G emitted tokens, final hidden states, exit logits, K/V rows and
spot-checked in-flight slot states.  The oracle values are position-keyed quantities of plain greedy decode, stored by
tests/golden/fullsize_golden.py (which calls only oracle/), or computed live with SPD_FULL_TIER=live.  The PDM, which
greedy decode does not define, is recomputed LIVE from the kernel's own slot vectors with the oracle's operations.
"""
from __future__ import annotations

import dataclasses
import importlib.util
import os

import numpy as np

import oracle as ora
import spd_inputs as si
from tests._parity import rel_err

_spec = importlib.util.spec_from_file_location("fullsize_golden", os.path.join(os.path.dirname(__file__), "golden",
                                                                              "fullsize_golden.py"))
fullsize_golden = importlib.util.module_from_spec(_spec)
_spec.loader.exec_module(fullsize_golden)

LIVE = os.environ.get("SPD_FULL_TIER", "") == "live"


def golden_for(name: str) -> dict:
    if LIVE:
        if name in ("9b_n4", "9b_n16"):
            if not hasattr(golden_for, "_pair"):
                golden_for._pair = fullsize_golden.compute_9b_pair()
            return golden_for._pair[name]
        return fullsize_golden.compute(name)
    return fullsize_golden.load(name)


@dataclasses.dataclass
class TierReport:
    tokens: int = 0
    cycles: int = 0
    accepts: int = 0
    rejects: int = 0
    ties: int = 0
    argmaxes: int = 0
    max_hfin_err: float = 0.0
    max_logit_err: float = 0.0        # relative to max|logit| (C-2.18)
    max_logit_abs: float = 0.0
    max_slot_err: float = 0.0
    slots_checked: int = 0
    max_pdm_err: float = 0.0
    pdm_checked: int = 0
    kv_flip: float = 0.0
    min_margin: float = 1.0

    def summary(self) -> str:
        return (f"tokens={self.tokens} cycles={self.cycles} acc/rej={self.accepts}/{self.rejects} ties={self.ties} of "
                f"{self.argmaxes} argmaxes hfin={self.max_hfin_err:.2e} logits={self.max_logit_err:.2e} (abs "
                f"{self.max_logit_abs:.2e}) slots={self.max_slot_err:.2e} ({self.slots_checked}) pdm={self.max_pdm_err:.2e} "
                f"({self.pdm_checked}) kvflip={self.kv_flip:.2e} min_margin={self.min_margin:.2e}")


def _bf16_close(got_bits, want_bits, what, tol, rep: TierReport):
    g = si.bf16_bits_to_f32(got_bits).astype(np.float64)
    o = si.bf16_bits_to_f32(want_bits).astype(np.float64)
    lim = 2.0 ** -7 * np.abs(o) + tol * np.max(np.abs(o))
    assert np.all(np.abs(g - o) <= lim), what
    rep.kv_flip = max(rep.kv_flip, float(np.mean(g != o)))


def _judge(g, i, token, logits_gpu, rep: TierReport, tol, what):
    """The CUDA path's token for position P + i against the oracle's tokens[i].  Exact: the token is the argmax of the
    CUDA path's own logits.  Measured: the logit difference on the stored entries (2048 samples + the oracle's top 32).
    A different token is a tie only if its ORACLE logit is within 3 x the measured difference of the oracle's maximum."""
    idx = np.concatenate([g["logit_idx"], g["top_idx"][i]])
    want = np.concatenate([g["logit_val"][i], g["top_val"][i]]).astype(np.float64)
    maxabs = float(g["logit_maxabs"][i])
    d = float(np.max(np.abs(logits_gpu[idx].astype(np.float64) - want)))
    rep.max_logit_abs = max(rep.max_logit_abs, d)
    rep.max_logit_err = max(rep.max_logit_err, d / maxabs)
    assert d / maxabs <= tol, f"{what}: logits differ by {d / maxabs:.2e} of max|logit|"
    assert int(np.argmax(logits_gpu)) == token, f"{what}: token {token} is not the argmax of the CUDA path's own logits"
    rep.argmaxes += 1
    rep.min_margin = min(rep.min_margin, float(g["top_val"][i][0] - g["top_val"][i][1]) / maxabs)
    want_tok = int(g["tokens"][i])
    if token == want_tok:
        return True
    band = 3.0 * rep.max_logit_abs + 1e-6 * maxabs
    where = np.where(g["top_idx"][i] == token)[0]
    assert len(where) and float(g["top_val"][i][0] - g["top_val"][i][where[0]]) <= band, \
        f"{what}: token {token} != oracle {want_tok} (outside the measured band {band:.2e})"
    rep.ties += 1
    return False


def oracle_tier(eng, shape, w, g, first, G=None, p=0.8, seed=3, tol=1e-2, pdm_every=4) -> TierReport:
    """`eng` has just prefilled the config's full prompt (DEBUG_LOGITS on) and returned `first`."""
    rep = TierReport()
    n, L, P, d = shape.n_stages, shape.n_layers, int(g["prompt_len"]), shape.d_model
    per = L // n
    G = len(g["tokens"]) - 1 if G is None else G
    h0 = int(g["hfin_pos0"])

    def hfin_check(pos):
        e = rel_err(eng.hfin(pos), g["hfin"][pos - h0])
        rep.max_hfin_err = max(rep.max_hfin_err, e)
        assert e <= tol, f"final hidden state of position {pos}: rel err {e:.2e}"

    # ---- the prefill result -------------------------------------------------------------------------------------
    for pos in range(h0, P):
        hfin_check(pos)
    for li, layer in enumerate(g["kv_layers"]):
        K, V = eng.kv(int(layer), 0, P), eng.kv(int(layer), 1, P)
        deep = layer > 0
        _bf16_close(K[g["kv_pos"]], g["k_rows"][li], f"layer {layer} K rows", 5e-3 if deep else 1e-4, rep)
        _bf16_close(V[g["kv_pos"]], g["v_rows"][li], f"layer {layer} V rows", 5e-3 if deep else 1e-4, rep)
    if not _judge(g, 0, first, eng.last("exit_logits"), rep, tol, "first token"):
        eng.rollback(P, int(g["tokens"][0]))                   # a measured tie: follow the oracle
    # ---- G tokens of SPD at forced acceptance p, compared position by position -----------------------------------
    truth = g["tokens"].astype(np.int32)
    eng.set_forced(truth, p, seed)
    trace_at = {int(pos): j for j, pos in enumerate(g["trace_pos"])}
    depth_of = {int(b) // per: j for j, b in enumerate(g["trace_layers"])}
    while rep.tokens < G:
        fill0, c0, slots0 = eng.ring()
        r = eng.step()
        rep.cycles += 1
        assert r.fill == fill0
        if not r.draft_forced:
            assert int(np.argmax(eng.last("pdm_logits"))) == r.draft_token, "draft is not the argmax of the CUDA PDM logits"
        # the PDM is a pure function of its n slot vectors: recomputed here by the oracle's operations from the kernel's
        # own slots; the slots themselves are the pre-step states (checked below as slot states / final hidden states)
        if rep.cycles % pdm_every == 1:
            feat = eng.last("pdm_feat")
            u = ora.op_gemv(w["pdm_proj"], feat)
            e = rel_err(eng.last("pdm_prenorm"), u)
            lp = ora.op_gemv(w["embed"], ora.op_rmsnorm(u, w["pdm_norm"], shape.rms_eps))
            e = max(e, rel_err(eng.last("pdm_logits"), lp))
            rep.max_pdm_err = max(rep.max_pdm_err, e)
            rep.pdm_checked += 1
            assert e <= 1e-3, f"cycle {rep.cycles}: PDM vs the oracle's operations on the same slots: {e:.2e}"
            p_new = slots0[0][1]
            for j in range(n):                                  # slot j = position p_new - j (C-2.2, C-2.4)
                q = p_new - j
                if not (j < fill0) and h0 <= q < c0:
                    e = rel_err(feat[j * d:(j + 1) * d], g["hfin"][q - h0])
                    assert e <= tol, f"cycle {rep.cycles}: warm-up slot {j} is not Hfin[{q}] ({e:.2e})"
        if r.exited:
            pos = r.committed_len - 1                           # the exited token's position; y decides position pos + 1
            i = pos + 1 - P
            hfin_check(pos)
            same = _judge(g, i, r.emitted_token, eng.last("exit_logits"), rep, tol, f"position {pos + 1}")
            rep.tokens += 1
            rep.accepts += r.accepted
            rep.rejects += 1 - r.accepted
            if not same:
                eng.rollback(pos + 1, int(g["tokens"][i]))      # a measured tie: follow the oracle
                continue
            if not r.accepted:
                assert np.all(eng.kv_len() == r.committed_len) and r.discarded == r.fill - 1
        # spot-checked slot states: a CORRECT in-flight token (behind correct ones) at depth k holds O-AR's residual stream after layer
        # k L/n - 1 at its position (SURVEY C-3)
        _, _, slots = eng.ring()
        right = [bool(o) and P <= q <= P + G and t == int(g["tokens"][q - P]) for o, q, t in slots]
        for k in range(1, n):
            occ, pos, tok = slots[k]
            # ... and so must every older in-flight token be: its K/V rows are part of this token's context
            if occ and pos in trace_at and k in depth_of and all(right[j] for j in range(k, n) if slots[j][0]):
                e = rel_err(eng.hidden(k), g["trace"][trace_at[pos], depth_of[k]])
                rep.max_slot_err = max(rep.max_slot_err, e)
                rep.slots_checked += 1
                assert e <= tol, f"slot state at depth {k}, position {pos}: rel err {e:.2e}"
    eng.set_forced(None, -1.0, 0)
    return rep
