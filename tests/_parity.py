"""GPU-vs-oracle parity harness (used by the -m gpu tests and __graft_entry__.smoke()).

Runs the CUDA library and the CPU oracle on the same seeded inputs, cycle by cycle, and compares:
step results (token ids, accept bits, fill, committed length: exact), per-depth hidden states, PDM
pre-norm vector, logits, KV lengths (exact) and KV rows.

Token exactness and ties.  The CUDA path accumulates in fp32, the oracle
in fp64; through 32 random-init layers that difference grows to ~1e-3 of the logit scale, while the
top-1/top-2 gap of 151 936 near-i.i.d. logits is below that for a small share of the argmaxes.  Protocol:
(1) every CUDA token must be the argmax (lowest index) of the CUDA path's OWN logit vector — exact;
(2) that vector must match the oracle's within the tensor tolerance;
(3) where the two argmaxes still differ, the CUDA token is adopted only if its ORACLE logit lies within
    band = 3 x the largest |gpu - oracle| logit difference MEASURED so far in the run (not the asserted
    tolerance) of the oracle's maximum; the oracle then follows that token (ora_step_follow) so every later
    cycle is still compared exactly.  Adoptions are counted (verify_ties / pdm_ties) and bounded by
    assert_ties(): zero whenever the smallest top-1/top-2 margin of the run exceeds twice the measured logit
    error, else a small share of the argmaxes.  Any other token difference is a failure.
"""
from __future__ import annotations

import dataclasses

import numpy as np

import spd_inputs as si
from oracle import Oracle

CONTRACT = 2e-2     # north_star: hidden states and logits within max relative error 2e-2


def rel_err(a, b) -> float:
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    den = float(np.max(np.abs(b)))
    return float(np.max(np.abs(a - b)) / (den if den > 0 else 1.0))


@dataclasses.dataclass
class Report:
    status: str = "ok"            # "ok" | "fail"
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
    verify_ties: int = 0
    pdm_ties: int = 0
    argmaxes: int = 0             # greedy decisions compared (first token + one per PDM pass + one per exit)
    max_logit_abs_err: float = 0.0
    tokens: list = dataclasses.field(default_factory=list)

    def summary(self) -> str:
        return (f"{self.status} steps={self.steps} emitted={self.emitted} acc/rej={self.accepts}/{self.rejects} "
                f"hidden={self.max_hidden_err:.2e} pdm={self.max_pdm_err:.2e} logits={self.max_logit_err:.2e} "
                f"kvflip={self.kv_flip_frac:.2e} min_margin={self.min_margin:.2e} "
                f"ties(verify/pdm)={self.verify_ties}/{self.pdm_ties} of {self.argmaxes} argmaxes "
                f"logit_abs={self.max_logit_abs_err:.2e} {self.detail}")


def assert_ties(rep: "Report", share: float = 0.05):
    """north_star: "emitted token ids exact".  Zero adoptions wherever the run's smallest top-1/top-2 margin exceeds
    twice the measured logit error (then no argmax can legitimately flip); otherwise at most `share` of the argmaxes
    (>= 1).  Both quantities are relative to max|logit| (C-2.18 metric)."""
    ties = rep.verify_ties + rep.pdm_ties
    if rep.min_margin > 2.0 * rep.max_logit_err:
        assert ties == 0, f"{ties} tie adoptions although min margin {rep.min_margin:.2e} > 2 x logit error {rep.max_logit_err:.2e}"
    else:
        assert ties <= max(1, int(share * rep.argmaxes)), f"{ties} tie adoptions in {rep.argmaxes} argmaxes"


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


def set_engine(gpu, engine):
    """engine: None (library default), 0 / 1 / 2, or (2, chains) = engine 2 with SPD_OPT_CHAINS = chains."""
    from paper_2605_30852_b200 import OPT
    if engine is None:
        return
    if isinstance(engine, tuple):
        gpu.set_option(OPT.ENGINE, engine[0])
        gpu.set_option(OPT.CHAINS, engine[1])
    else:
        gpu.set_option(OPT.ENGINE, engine)


def run_parity(shape, weights_np, dev_weights, prompt, n_tokens, forced=None, engine=None, tensor_every=1,
               tensor_tol=CONTRACT, check_logits=True, prefill_block=16, max_seq=None, gpu=None, prefill_mode=None) -> Report:
    """forced = (truth tokens, p, seed) or None (the PDM's own drafts).  tensor_tol bounds hidden states,
    the PDM vector and logits (C-2.18 metric); the tie band is 3 x the measured logit difference (module doc)."""
    from paper_2605_30852_b200 import SPD, OPT
    rep = Report()
    n = shape.n_stages
    ms = max_seq or (len(prompt) + n_tokens * (n + 1) + 2 * n + 8)
    ora = Oracle(shape, weights_np, max_seq=ms)
    own = gpu is None
    if own:
        gpu = SPD(shape, dev_weights, max_seq=ms)

    def fail(msg):
        rep.status, rep.detail = "fail", msg
        return rep

    try:
        set_engine(gpu, engine)
        if prefill_mode is not None:             # 1: batched tensor-core prefill (the default), 0: through the decode kernel
            gpu.set_option(OPT.PREFILL, prefill_mode)
        gpu.set_option(OPT.DEBUG_LOGITS, 1)      # the measured logit difference sets the tie band
        fo = ora.prefill(prompt, block=prefill_block)
        fg = gpu.prefill(prompt)
        gap, mx = ora.margin(0)
        rep.min_margin = gap / mx
        lg_g, lg_o = gpu.last("exit_logits"), ora.last("exit_logits")
        delta_run = float(np.max(np.abs(lg_g.astype(np.float64) - lg_o)))
        maxabs = float(mx)
        rep.max_logit_abs_err = delta_run
        rep.max_logit_err = delta_run / maxabs
        rep.argmaxes = 1
        if int(np.argmax(lg_g)) != fg:
            return fail(f"first token {fg} is not the argmax of the CUDA path's own logits ({int(np.argmax(lg_g))})")
        if rep.max_logit_err > tensor_tol:
            return fail(f"prefill logits rel err {rep.max_logit_err:.3e}")
        band = 3.0 * delta_run + 1e-6 * maxabs
        P = len(prompt)
        e = rel_err(gpu.hfin(P - 1), ora.hfin(P - 1))
        rep.max_hidden_err = max(rep.max_hidden_err, e)
        if e > tensor_tol:
            return fail(f"prefill final hidden state rel err {e:.3e}")
        if fo != fg:
            lg = ora.last("exit_logits")
            if lg[fo] - lg[fg] <= band:
                rep.verify_ties += 1
                ora.rollback(P, fg)          # both are valid first tokens at the logit tolerance: follow the GPU
            else:
                return fail(f"first token {fg} != oracle {fo} (margin {gap / mx:.2e})")
        rep.tokens.append(fg)
        if not np.array_equal(gpu.kv_len(), ora.kv_len()):
            return fail("KV lengths differ after prefill")
        if not kv_compare(gpu, ora, sorted({0, shape.n_layers // 2, shape.n_layers - 1}), P, rep, tensor_tol):
            return rep
        if forced is not None:
            truth, p, seed = forced
            ora.set_forced(truth, p, seed)
            gpu.set_forced(truth, p, seed)
        v0 = rep.verify_ties
        while ora.emitted < n_tokens:
            rg = gpu.step()
            band = 3.0 * delta_run + 1e-6 * maxabs
            ro = ora.step_follow(-1 if rg.draft_forced else rg.draft_token, rg.emitted_token if rg.exited else -1, band)
            rep.steps += 1
            rep.argmaxes += 1 + (1 if rg.exited else 0)
            # (1) the CUDA tokens are the argmax (lowest index) of the CUDA path's own logit vectors; (2) the measured
            # logit difference of this cycle widens the band of the following cycles
            lp_g, lp_o = gpu.last("pdm_logits"), ora.last("pdm_logits")
            if not rg.draft_forced and int(np.argmax(lp_g)) != rg.draft_token:
                return fail(f"step {rep.steps}: draft {rg.draft_token} is not the argmax of the CUDA PDM logits")
            d = float(np.max(np.abs(lp_g.astype(np.float64) - lp_o)))
            maxabs = max(maxabs, float(np.max(np.abs(lp_o))))
            rep.max_logit_err = max(rep.max_logit_err, rel_err(lp_g, lp_o))
            if rg.exited:
                le_g, le_o = gpu.last("exit_logits"), ora.last("exit_logits")
                if int(np.argmax(le_g)) != rg.emitted_token:
                    return fail(f"step {rep.steps}: emitted {rg.emitted_token} is not the argmax of the CUDA exit logits")
                d = max(d, float(np.max(np.abs(le_g.astype(np.float64) - le_o))))
                maxabs = max(maxabs, float(np.max(np.abs(le_o))))
                rep.max_logit_err = max(rep.max_logit_err, rel_err(le_g, le_o))
            delta_run = max(delta_run, d)
            rep.max_logit_abs_err = delta_run
            if rep.max_logit_err > tensor_tol:
                return fail(f"step {rep.steps}: logits rel err {rep.max_logit_err:.3e} > {tensor_tol}")
            vt, pt = ora.ties()
            rep.verify_ties, rep.pdm_ties = v0 + vt, pt
            if tuple(ro) != tuple(rg):
                gv, mv = ora.margin(0)
                gp, mp = ora.margin(1)
                return fail(f"step {rep.steps}: gpu {tuple(rg)} != oracle {tuple(ro)} "
                            f"(verify margin {gv / mv:.2e}, PDM margin {gp / mp:.2e}, band {band:.1e} abs = "
                            f"{band / maxabs:.1e} of max|logit|)")
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
                    return fail(f"step {rep.steps}: ring fill/committed differ")
                for i in range(ora.fill):
                    pos, tok, k, h = ora.ring(i)
                    if slots[k] != (1, pos, tok):
                        return fail(f"step {rep.steps}: depth {k} holds {slots[k]}, oracle ({pos},{tok})")
                    rep.max_hidden_err = max(rep.max_hidden_err, rel_err(gpu.hidden(k), h))
                rep.max_pdm_err = max(rep.max_pdm_err, rel_err(gpu.last("pdm_prenorm"), ora.last("pdm_prenorm")))
                if not np.array_equal(gpu.kv_len(), ora.kv_len()):
                    return fail(f"step {rep.steps}: KV lengths differ")
                worst = max(rep.max_hidden_err, rep.max_pdm_err, rep.max_logit_err)
                if worst > tensor_tol:
                    return fail(f"step {rep.steps}: tensor rel err {worst:.3e} > {tensor_tol}")
        kv_compare(gpu, ora, sorted({0, shape.n_layers - 1}), ora.committed_len, rep, tensor_tol)
        return rep
    finally:
        ora.close()
        if own:
            gpu.close()


# ------------------------------------------------------------------ sampling verification (NEXT-2) ----

@dataclasses.dataclass
class SamplingReport:
    status: str = "ok"
    detail: str = ""
    steps: int = 0
    emitted: int = 0
    accepts: int = 0
    rejects: int = 0
    max_logit_abs_err: float = 0.0
    max_prob_err: float = 0.0
    max_hidden_err: float = 0.0
    ties: tuple = (0, 0, 0, 0)       # hints adopted: support, draft, accept, replacement
    exact_rounds: int = 0
    prefiltered: int = 0             # selections served by the fused head pass's threshold list (no scan)
    tokens: list = dataclasses.field(default_factory=list)

    def summary(self) -> str:
        return (f"{self.status} steps={self.steps} emitted={self.emitted} acc/rej={self.accepts}/{self.rejects} "
                f"logit_abs={self.max_logit_abs_err:.2e} prob={self.max_prob_err:.2e} hidden={self.max_hidden_err:.2e} "
                f"ties(support/draft/accept/repl)={self.ties} exact_rounds={self.exact_rounds} prefiltered={self.prefiltered} {self.detail}")


def _dist_close(g, o, delta):
    """Same support; probabilities within what a logit difference `delta` allows (|dp| <= (e^(2 delta) - 1) p)."""
    gi, gp = g
    if not np.array_equal(gi, o.ids):
        return False, float("inf")
    err = np.abs(gp.astype(np.float64) - o.p.astype(np.float64))
    lim = np.expm1(2.0 * delta) * o.p.astype(np.float64) + 2e-7
    return bool(np.all(err <= lim)), float(err.max()) if err.size else 0.0


def run_sampling_parity(shape, weights_np, dev_weights, prompt, n_tokens, temperature, top_k, seed, engine=None,
                        tensor_tol=CONTRACT, max_seq=None, max_steps=None, greedy_steps=0) -> SamplingReport:
    """GPU vs oracle in sampling mode, cycle by cycle.  Exact: step results (tokens, accept bits, fill,
    committed length), uniforms, supports, KV lengths.  Within tolerance: logits (tensor_tol, C-2.18),
    probabilities (bounded by the measured logit difference), hidden states.

    Decisions taken on floating point (top-k membership at the k-th/k+1-th boundary, inverse-CDF draws, the
    accept test) may legitimately differ where the uniform / the logit lies within the measured logit
    difference of the decision boundary.  The oracle is told what the CUDA path decided
    (ora_step_sample_follow) and adopts it ONLY in that case (band = 3 x the largest logit difference measured
    so far; the adoptions are counted in `ties`); any other difference fails."""
    from paper_2605_30852_b200 import SPD, OPT
    rep = SamplingReport()
    n = shape.n_stages
    ms = max_seq or (len(prompt) + n_tokens * (n + 1) + 2 * n + 8)
    ora = Oracle(shape, weights_np, max_seq=ms)
    gpu = SPD(shape, dev_weights, max_seq=ms)

    def fail(msg):
        rep.status, rep.detail = "fail", msg
        return rep

    try:
        set_engine(gpu, engine)
        if greedy_steps:      # greedy prefill + cycles first; sampling is switched on with tokens in flight
            gpu.set_option(OPT.DEBUG_LOGITS, 1)
        else:
            ora.set_sampling(temperature, top_k, seed)
            gpu.set_sampling(temperature, top_k, seed)
        fo = ora.prefill(prompt, block=16)
        fg = gpu.prefill(prompt)
        lo, lg = ora.last("exit_logits"), gpu.last("exit_logits")
        delta_run = float(np.max(np.abs(lo.astype(np.float64) - lg)))
        maxabs = float(np.max(np.abs(lo)))
        rep.max_logit_abs_err = delta_run
        if delta_run > tensor_tol * maxabs:
            return fail(f"prefill logits differ by {delta_run:.3e} (max|logit| {maxabs:.3f})")
        if greedy_steps:
            if fo != fg:
                return fail(f"greedy first token {fg} vs oracle {fo}")
            for i in range(greedy_steps):
                rg, ro = gpu.step(), ora.step()
                if tuple(rg) != tuple(ro):
                    return fail(f"greedy step {i + 1}: gpu {tuple(rg)} != oracle {tuple(ro)}")
            ora.set_sampling(temperature, top_k, seed)
            gpu.set_sampling(temperature, top_k, seed)
        else:
            orec, grec = ora.sample_record(), gpu.sample_record()
            if grec["u_resid"] != orec["u_resid"]:
                return fail("first-token uniform differs")
            ok, perr = _dist_close(grec["target"], orec["target"], delta_run)
            if fo != fg or not ok:
                return fail(f"first token {fg} vs oracle {fo}, distributions close: {ok} (prob err {perr:.2e})")
            rep.max_prob_err = perr
        rep.tokens.append(fg)
        limit = max_steps or 10 ** 9
        while ora.emitted < n_tokens and rep.steps < limit:
            rg = gpu.step()
            grec = gpu.sample_record()
            band = 3.0 * delta_run + 1e-6 * maxabs
            ro = ora.step_sample_follow(draft_ids=grec["draft"][0], verify_ids=grec["target"][0] if rg.exited else None,
                                        draft_token=rg.draft_token, accepted=rg.accepted if rg.exited else -1,
                                        emitted_token=rg.emitted_token if rg.exited and not rg.accepted else -1,
                                        logit_band=band, prob_eps=4.0 * band)
            orec = ora.sample_record()
            rep.steps += 1
            rep.ties = orec["ties"]
            rep.exact_rounds += grec["exact_rounds"]
            rep.prefiltered += grec["prefiltered"]
            # logits first: they bound everything else
            d = float(np.max(np.abs(ora.last("pdm_logits").astype(np.float64) - gpu.last("pdm_logits"))))
            if ro.exited:
                d = max(d, float(np.max(np.abs(ora.last("exit_logits").astype(np.float64) - gpu.last("exit_logits")))))
                maxabs = max(maxabs, float(np.max(np.abs(ora.last("exit_logits")))))
            rep.max_logit_abs_err = max(rep.max_logit_abs_err, d)
            if d > tensor_tol * maxabs:
                return fail(f"step {rep.steps}: logits differ by {d:.3e} (max|logit| {maxabs:.3f})")
            if tuple(ro) != tuple(rg):
                return fail(f"step {rep.steps}: gpu {tuple(rg)} != oracle {tuple(ro)} (band {band:.2e}, "
                            f"u = {orec['u_draft']:.7f}/{orec['u_accept']:.7f}/{orec['u_resid']:.7f})")
            for key in ("u_draft", "u_accept", "u_resid"):
                if float(grec[key]) != float(orec[key]):
                    return fail(f"step {rep.steps}: {key} gpu {grec[key]} != oracle {orec[key]}")
            ok, perr = _dist_close(grec["draft"], orec["draft"], max(d, delta_run))
            if not ok:
                return fail(f"step {rep.steps}: draft distribution differs (prob err {perr:.2e})")
            rep.max_prob_err = max(rep.max_prob_err, perr)
            if ro.exited:
                ok, perr = _dist_close(grec["target"], orec["target"], max(d, delta_run))
                if not ok or grec["succ_token"] != orec["succ_token"]:
                    return fail(f"step {rep.steps}: target distribution / judged token differs (prob err {perr:.2e})")
                rep.max_prob_err = max(rep.max_prob_err, perr)
                if abs(grec["succ_q"] - orec["succ_q"]) > np.expm1(2 * max(d, delta_run)) * orec["succ_q"] + 2e-7:
                    return fail(f"step {rep.steps}: stored draft probability of the judged token differs")
                rep.emitted += 1
                rep.tokens.append(ro.emitted_token)
                rep.accepts += ro.accepted
                rep.rejects += 1 - ro.accepted
            delta_run = max(delta_run, d)
            fill, c, slots = gpu.ring()
            if fill != ora.fill or c != ora.committed_len:
                return fail(f"step {rep.steps}: ring fill/committed differ")
            for i in range(ora.fill):
                pos, tok, k, h = ora.ring(i)
                if slots[k] != (1, pos, tok):
                    return fail(f"step {rep.steps}: depth {k} holds {slots[k]}, oracle ({pos},{tok})")
                rep.max_hidden_err = max(rep.max_hidden_err, rel_err(gpu.hidden(k), h))
            if rep.max_hidden_err > tensor_tol:
                return fail(f"step {rep.steps}: hidden rel err {rep.max_hidden_err:.3e}")
            if not np.array_equal(gpu.kv_len(), ora.kv_len()):
                return fail(f"step {rep.steps}: KV lengths differ")
        return rep
    finally:
        ora.close()
        gpu.close()
