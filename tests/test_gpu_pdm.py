"""The paper's Pipeline Draft Module on the device against the oracle (-m gpu), through the C ABI.

Cycle by cycle, both engines: step results (draft token from the reduced vocabulary through vocab_map, accept bits,
emitted tokens, fills, committed length) exact under the measured-band tie protocol of tests/_parity.py; the PDM's
logits and last hidden state, the rows it refreshed (first position, count, F), the target's hidden states and exit
logits within tolerance; the anchors H^b captured by the target's forward (prompt positions through either prefill
path, generated positions through the cycle kernel); at the end the PDM's own KV cache rows of every layer within one
bf16 ulp.  Shapes: tiny at n = 1, 2, 4, 8 (forced acceptance mixes accepts and rejects), a head_dim-128 decoder, and
the 4B-class dimensions with a short prompt.
"""
import numpy as np
import pytest

import spd_inputs as si
from oracle import Oracle
from tests._parity import rel_err
from tests._util import shape_of

pytestmark = pytest.mark.gpu


def run_pdm_parity(shape, w, pw, prompt, n_tokens, engine, forced_p=None, tol=5e-3, prefill_mode=None):
    """tol bounds the target's tensors; the PDM's own tensors get 4 x tol: its L_s layers sit on top of the target's
    hidden states (their fp32-vs-fp64 difference is its INPUT) and round their own K/V rows to bf16 once more — the CPU
    pin of the oracle against the float64 model shows the same factor (tests/test_oracle_pdm.py: 2e-2 on this init)."""
    import paper_2605_30852_b200 as spd
    ptol = 4.0 * tol
    n, P = shape.n_stages, len(prompt)
    ms = P + n_tokens * (n + 1) + 2 * n + 8
    ora = Oracle(shape, w, max_seq=ms)
    ora.attach_pdm(pw)
    gpu = spd.SPD(shape, spd.upload_weights(w), max_seq=ms)
    rep = dict(steps=0, emitted=0, accepts=0, rejects=0, ties=0, pdm_err=0.0, hidden_err=0.0, logit_err=0.0, delta=0.0)
    try:
        gpu.attach_pdm(spd.upload_pdm_weights(pw))
        gpu.set_option(spd.OPT.ENGINE, engine)
        gpu.set_option(spd.OPT.DEBUG_LOGITS, 1)
        if prefill_mode is not None:
            gpu.set_option(spd.OPT.PREFILL, prefill_mode)
        with pytest.raises(spd.SpdError):
            gpu.set_sampling(1.0, 50, 1)                      # greedy only (reading P-9)
        fo, fg = ora.prefill(prompt, block=16), gpu.prefill(prompt)
        lo, lg = ora.last("exit_logits"), gpu.last("exit_logits")
        delta, maxabs = float(np.max(np.abs(lg.astype(np.float64) - lo))), float(np.max(np.abs(lo)))
        assert delta <= tol * maxabs
        assert fg == fo or lo[fo] - lo[fg] <= 3 * delta, "first token"
        if fg != fo:
            ora.rollback(P, fg)
        B = ora.pdm_anchors()
        for pos in sorted({0, 1, P // 2, P - 1}):             # anchors of prompt positions (captured by the prefill)
            for i in range(len(B)):
                e = rel_err(gpu.anchor(pos, i), ora.pdm_anchor(pos, i))
                assert e <= tol, f"anchor H^{B[i]} of position {pos}: {e:.2e}"
        assert gpu.pdm_run()[2] == P                          # the prompt's full-depth PDM rows are built by spd_prefill
        if forced_p is not None:
            t = Oracle(shape, w, max_seq=ms)
            truth = np.array([t.prefill(prompt, block=16)] + [t.ar_step() for _ in range(n_tokens + n + 2)], np.int32)
            t.close()
            ora.set_forced(truth, forced_p, 5)
            gpu.set_forced(truth, forced_p, 5)
        vmap = pw["vocab_map"]
        while ora.emitted < n_tokens:
            c_before = ora.committed_len
            rg = gpu.step()
            band = 3.0 * delta + 1e-6 * maxabs
            ro = ora.step_follow(-1 if rg.draft_forced else rg.draft_token, rg.emitted_token if rg.exited else -1, band)
            rep["steps"] += 1
            pl_g, pl_o = gpu.pdm_last("logits"), ora.pdm_last("logits")
            if not rg.draft_forced:
                assert int(vmap[int(np.argmax(pl_g))]) == rg.draft_token, "draft is not vocab_map[argmax] of the CUDA PDM logits"
                assert rg.draft_token in set(vmap)
            d = float(np.max(np.abs(pl_g.astype(np.float64) - pl_o)))
            pm = float(np.max(np.abs(pl_o)))
            rep["pdm_err"] = max(rep["pdm_err"], d / pm, rel_err(gpu.pdm_last("hidden"), ora.pdm_last("hidden")))
            assert rep["pdm_err"] <= ptol, f"step {rep['steps']}: PDM logits / hidden rel err {rep['pdm_err']:.2e}"
            delta = max(delta, d)
            if rg.exited:
                le_g, le_o = gpu.last("exit_logits"), ora.last("exit_logits")
                assert int(np.argmax(le_g)) == rg.emitted_token
                delta = max(delta, float(np.max(np.abs(le_g.astype(np.float64) - le_o))))
                rep["logit_err"] = max(rep["logit_err"], rel_err(le_g, le_o))
            assert tuple(rg) == tuple(ro), f"step {rep['steps']}: gpu {tuple(rg)} != oracle {tuple(ro)} (band {band:.2e})"
            first_o, depths_o = ora.pdm_rows()
            first_g, rows_g, fin_g = gpu.pdm_run()
            assert fin_g == c_before
            if rep["steps"] > 1:                              # the oracle builds the prompt's rows lazily in its first cycle
                assert (first_g, rows_g) == (first_o, len(depths_o)) and rows_g <= n + 1
                e = rel_err(gpu.pdm_last("features"), ora.pdm_last("features"))
                assert e <= ptol, f"step {rep['steps']}: features g (Eq. 4) rel err {e:.2e}"
            if ro.exited:
                rep["emitted"] += 1
                rep["accepts"] += ro.accepted
                rep["rejects"] += 1 - ro.accepted
            fill, c, slots = gpu.ring()
            assert (fill, c) == (ora.fill, ora.committed_len)
            for i in range(ora.fill):
                pos, tok, k, h = ora.ring(i)
                assert slots[k] == (1, pos, tok)
                rep["hidden_err"] = max(rep["hidden_err"], rel_err(gpu.hidden(k), h))
            assert rep["hidden_err"] <= tol and rep["logit_err"] <= tol
            assert np.array_equal(gpu.kv_len(), ora.kv_len())
        vt, pt = ora.ties()
        rep["ties"] = vt + pt
        rep["delta"] = delta
        c = ora.committed_len
        for pos in (P, c - 1):                                # anchors of generated positions (captured by the cycle)
            for i in range(len(B)):
                assert rel_err(gpu.anchor(pos, i), ora.pdm_anchor(pos, i)) <= tol
        flips = 0.0
        for l in range(pw["n_layers"]):                       # the PDM's own cache: final rows of every layer
            for which in (0, 1):
                go = si.bf16_bits_to_f32(gpu.pdm_kv(l, which, c)).astype(np.float64)
                oo = si.bf16_bits_to_f32(ora.pdm_kv(l, which, c)[0]).astype(np.float64)
                assert np.all(np.abs(go - oo) <= 2.0 ** -7 * np.abs(oo) + ptol * np.abs(oo).max()), f"PDM layer {l} cache"
                flips = max(flips, float(np.mean(go != oo)))
        rep["kvflip"] = flips
        return rep
    finally:
        ora.close()
        gpu.close()


@pytest.mark.parametrize("engine", [0, 1, 2])
@pytest.mark.parametrize("n,pdm_layers,forced_p", [(1, 1, None), (2, 2, None), (4, 3, 0.7), (8, 2, 0.8), (4, 1, 1.0)])
def test_tiny_paper_pdm(engine, n, pdm_layers, forced_p):
    shape = shape_of("tiny", n)
    w = si.make_weights(shape, seed=1234, std=0.08, random_gains=True)
    pw = si.make_pdm_weights(shape, pdm_layers, 300, seed=1234, std=0.08, random_gains=True)
    rep = run_pdm_parity(shape, w, pw, si.make_prompt(shape, 1, 40), 30, engine, forced_p)
    print(f"tiny n={n} Ls={pdm_layers} p={forced_p} engine={engine}:", rep)
    assert rep["ties"] <= 1
    if forced_p is not None and forced_p < 1.0:
        assert rep["accepts"] > 0 and rep["rejects"] > 0


@pytest.mark.parametrize("prefill_mode", [0, 1])
def test_baseline_init_and_both_prefill_paths(prefill_mode):
    shape = shape_of("tiny", 2)
    w = si.make_weights(shape, seed=1234)
    pw = si.make_pdm_weights(shape, 2, 1024, seed=1234)          # V_s = V: the map is the identity
    assert np.array_equal(pw["vocab_map"], np.arange(shape.vocab))
    rep = run_pdm_parity(shape, w, pw, si.make_prompt(shape, 1), 40, 1, None, tol=1e-3, prefill_mode=prefill_mode)
    print(f"tiny baseline init, prefill mode {prefill_mode}:", rep)
    assert rep["ties"] == 0


def test_head_dim_128_and_ragged_rows():
    shape = si.ModelShape("mid", 512, 8, 4, 8, 2, 128, 1024, 2048, 200, 24, ())
    w = si.make_weights(shape, seed=1234, std=0.04)
    pw = si.make_pdm_weights(shape, 2, 777, seed=1234, std=0.04)
    rep = run_pdm_parity(shape, w, pw, si.make_prompt(shape, 3, 200), 24, 1, 0.75, tol=2e-3)
    print("mid hd128:", rep)
    assert rep["ties"] <= 1 and rep["rejects"] > 0


@pytest.mark.timeout(900)
@pytest.mark.parametrize("name,pdm_layers", [("4b_n4", 2), ("9b_n16", 1)])
def test_full_model_dims_paper_pdm(name, pdm_layers):
    """The 4B / 9B-class dimensions (d 2560 / 4096, F 9728 / 12288) with a short prompt and a 32000-entry head."""
    shape = si.CONFIGS[name]
    w = si.make_weights(shape, seed=1234)
    pw = si.make_pdm_weights(shape, pdm_layers, 32000, seed=1234)
    rep = run_pdm_parity(shape, w, pw, si.make_prompt(shape, 1234, 24), 10, 1, 0.7, tol=1e-2)
    print(name, rep)
    assert rep["ties"] <= 1


@pytest.mark.parametrize("engine", [0, 1, 2])
def test_external_rollback_and_second_prefill_with_the_paper_pdm(engine):
    """spd_rollback rewinds the PDM's final-row count F with the committed length (rows above are rebuilt by the next
    draft); a second spd_prefill on the same context starts a new sequence.  Step results against the oracle."""
    import paper_2605_30852_b200 as spd
    shape = shape_of("tiny", 4)
    w = si.make_weights(shape, seed=1234, std=0.08, random_gains=True)
    pw = si.make_pdm_weights(shape, 2, 300, seed=1234, std=0.08, random_gains=True)
    ora = Oracle(shape, w, max_seq=400)
    ora.attach_pdm(pw)
    gpu = spd.SPD(shape, spd.upload_weights(w), max_seq=400)
    gpu.attach_pdm(spd.upload_pdm_weights(pw))
    gpu.set_option(spd.OPT.ENGINE, engine)
    rng = np.random.default_rng(5)
    try:
        for seq in range(2):
            prompt = si.make_prompt(shape, 11 + seq, 37 + 20 * seq)
            assert gpu.prefill(prompt) == ora.prefill(prompt, block=8)
            for rnd in range(4):
                for _ in range(9):
                    a, b = gpu.step(), ora.step_follow(-1, -1, 0.0)
                    assert tuple(a) == tuple(b), (seq, rnd)
                    assert gpu.pdm_run()[2] <= ora.committed_len
                c = ora.committed_len
                new_len, tok = int(c - rng.integers(0, 4)), int(rng.integers(0, shape.vocab))
                gpu.rollback(new_len, tok)
                assert ora.rollback(new_len, tok) == 0
                assert gpu.pdm_run()[2] <= new_len
                fill, cc, slots = gpu.ring()
                assert (fill, cc, slots[0]) == (1, new_len, (1, new_len, tok))
    finally:
        ora.close()
        gpu.close()
