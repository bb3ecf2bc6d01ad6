"""Pins for the oracle's decoder and SPD state machine.  CPU only.

What fixes the oracle here is NOT the oracle itself: a separately written float64 no-cache numpy model
(library matmul/softmax, complex-form RoPE), the three facts the paper's definition fixes
(n=1 == autoregressive; greedy SPD is lossless; rollback leaves KV as if the rejected
tokens never ran), the depth staircase and closed-form step counts.
"""
import numpy as np
import pytest

import spd_inputs as si
from oracle import Oracle, op_splitmix64
from oracle.nocache_ref import forward_nocache, pdm_ref
from tests._util import TINY, ar_tokens, shape_of, weights

P = TINY.prompt_len
G = TINY.gen_len
PROMPT = si.make_prompt(TINY, 1)


def new_oracle(n=None, **wkw):
    shape = shape_of("tiny", n)
    return Oracle(shape, weights("tiny", n, **wkw), max_seq=1024)


# ------------------------------------------------------------------ O-AR vs the no-cache model ---

# (init, logits/hidden tolerance, allowed fraction of K/V entries on the other side of a bf16 rounding
# boundary).  With BASELINE.json's init (std 0.02, gains 1) the two models agree to ~5e-6.  The hot and
# attention-heavy test inits are far more sensitive: rounding K/V to bf16 turns an fp32-level difference
# delta into ~sqrt(delta * 2^-8) on the cache (a fraction delta/2^-8 of entries moves one bf16 ulp), and
# those inits feed that straight back through attention, so the floor there is ~1e-4, not 1e-6.
@pytest.mark.parametrize("wkw,tol,flips", [(dict(), 2e-3, 0.15), (dict(std=0.02, random_gains=False), 1e-4, 5e-3),
                                           (dict(attention_heavy=True), 2e-3, 0.15)],
                         ids=["hot", "baseline_init", "attention_heavy"])
def test_ar_decode_matches_nocache_float64_model(wkw, tol, flips):
    """Every emitted position: logits within tol (C-2.18 metric; 1e-4 at the BASELINE init) and argmax
    exact vs a whole-prefix recompute that shares no code with the C oracle; K/V rows and final hidden
    states too."""
    o = new_oracle(**wkw)
    w = weights("tiny", None, **wkw)
    toks = [o.prefill(PROMPT)]
    logits = [o.last("exit_logits")]
    for _ in range(G - 1):
        toks.append(o.ar_step())
        logits.append(o.last("exit_logits"))
    seq = np.concatenate([PROMPT, np.array(toks[:-1], dtype=np.int32)])
    ref = forward_nocache(TINY, w, seq)
    for i in range(G):
        r = ref["logits"][P - 1 + i]
        assert int(np.argmax(r)) == toks[i], f"token {i}"
        assert np.max(np.abs(logits[i] - r)) / np.max(np.abs(r)) < tol
    T = len(seq)
    assert o.committed_len == T
    for l in range(TINY.n_layers):
        for which, name in ((0, "k"), (1, "v")):
            got = si.bf16_bits_to_f32(o.kv(l, which, T)).astype(np.float64)
            want = ref[name][l]
            # bf16-exact but for rounding-boundary ulps (the oracle rounds fp32->bf16, the model f64->bf16)
            bad = np.abs(got - want) > 1e-12
            assert bad.mean() < flips
            # every entry within one bf16 ulp of itself plus the fp-level slack of the tensor
            assert np.all(np.abs(got - want) <= 2.0 ** -7 * np.abs(want) + tol * np.max(np.abs(want)))
    for pos in (0, P - 1, T - 1):
        assert np.max(np.abs(o.hfin(pos) - ref["final"][pos])) / np.max(np.abs(ref["final"][pos])) < tol


def test_blocked_prefill_is_bitwise_the_plain_prefill():
    a, b = new_oracle(), new_oracle()
    ya = a.prefill(PROMPT, block=1)
    yb = b.prefill(PROMPT, block=5)   # ragged: 32 = 6*5 + 2
    assert ya == yb
    assert np.array_equal(a.last("exit_logits"), b.last("exit_logits"))
    for l in range(TINY.n_layers):
        assert np.array_equal(a.kv(l, 0, P), b.kv(l, 0, P)) and np.array_equal(a.kv(l, 1, P), b.kv(l, 1, P))
    for pos in range(P):
        assert np.array_equal(a.hfin(pos), b.hfin(pos))


# ------------------------------------------------------------------ fact 1: n = 1 is AR ------------

def test_spd_with_one_stage_is_autoregressive_decode_bitwise():
    ar = new_oracle(1)
    sp = new_oracle(1)
    ar.prefill(PROMPT)
    sp.prefill(PROMPT)
    ar_toks = [ar.ar_step() for _ in range(G - 1)]
    sp_toks, log = sp.generate_spd(G)
    assert sp_toks == ar_toks
    assert len(log) == G - 1 and all(r.exited and r.fill == 1 for r in log)
    assert sp.committed_len == ar.committed_len
    assert np.array_equal(sp.kv_len(), ar.kv_len())
    T = ar.committed_len
    for l in range(TINY.n_layers):
        assert np.array_equal(sp.kv(l, 0, T), ar.kv(l, 0, T)) and np.array_equal(sp.kv(l, 1, T), ar.kv(l, 1, T))
    for pos in range(T):
        assert np.array_equal(sp.hfin(pos), ar.hfin(pos))


# ------------------------------------------------------------------ fact 2: lossless ---------------

def _draft_fn(mode, truth, vocab, rng):
    def fn(o):
        pos_new = o.ring(o.fill - 1)[0]
        t = truth[pos_new + 1 - P] if pos_new + 1 - P < len(truth) else 0
        if mode == "right":
            return t
        if mode == "wrong":
            return (t + 1) % vocab
        if mode == "random":
            return t if rng.random() < 0.5 else int(rng.integers(0, vocab))
        return -1  # the PDM's own token
    return fn


@pytest.mark.parametrize("n", [1, 2, 4, 8])
@pytest.mark.parametrize("mode", ["pdm", "right", "wrong", "random"])
def test_greedy_spd_is_lossless(n, mode):
    truth = ar_tokens("tiny", G + 16)
    o = new_oracle(n)
    first = o.prefill(PROMPT)
    assert first == truth[0]
    toks, log = o.generate_spd(G, _draft_fn(mode, truth, TINY.vocab, np.random.default_rng(n)))
    assert [first] + toks == list(truth[:G])
    assert o.emitted == 1 + sum(r.exited for r in log)          # N = 1 + #exit-steps (C-2.9)
    if mode == "right":
        assert len(log) == G + n - 2                             # first exit at step n, then one per step
        assert all(r.accepted for r in log if r.exited)
    if mode == "wrong" and n > 1:
        assert len(log) == (G - 1) * n                           # every token costs a full refill
        assert not any(r.accepted for r in log)


@pytest.mark.parametrize("n", [2, 4])
@pytest.mark.parametrize("p", [0.0, 0.4, 0.6, 0.8, 1.0])
def test_forced_acceptance_is_lossless_and_follows_the_integer_rule(n, p):
    truth = np.array(ar_tokens("tiny", G + 16), dtype=np.int32)
    o = new_oracle(n)
    first = o.prefill(PROMPT)
    seed = 7
    o.set_forced(truth, p, seed)
    toks, log = o.generate_spd(G)
    assert [first] + toks == list(truth[:G])
    thresh = int(np.floor(float(np.float32(p)) * 2.0 ** 53))
    for r in log:                                                # C-2.19, recomputed here in Python
        want = (op_splitmix64(seed + r.step_index) >> 11) < thresh
        assert bool(r.draft_forced) == want
    if p == 1.0:
        assert len(log) == G + n - 2 and all(r.accepted for r in log if r.exited)


# ------------------------------------------------------------------ fact 3: rollback identity ------

@pytest.mark.parametrize("n", [2, 4])
def test_rollback_leaves_kv_as_if_rejected_tokens_never_ran(n):
    truth = ar_tokens("tiny", G + 16)
    ar = new_oracle(n)
    ar.prefill(PROMPT)
    ar_kv = {}                                                   # AR cache after all tokens
    for _ in range(G + 8):
        ar.ar_step()
    T_ar = ar.committed_len
    for l in range(TINY.n_layers):
        ar_kv[l] = (ar.kv(l, 0, T_ar), ar.kv(l, 1, T_ar))
    o = new_oracle(n)
    o.prefill(PROMPT)
    rng = np.random.default_rng(3)
    fn = _draft_fn("random", truth, TINY.vocab, rng)
    rejects = 0
    while o.emitted < G:
        r = o.step(fn(o))
        if r.exited and not r.accepted:
            rejects += 1
            c = r.committed_len
            assert r.discarded == r.fill - 1
            assert np.all(o.kv_len() == c)                       # "truncate target KV caches"
            assert o.fill == 1 and o.ring(0)[:3] == (c, r.emitted_token, 0)
            for l in range(TINY.n_layers):
                assert np.array_equal(o.kv(l, 0, c), ar_kv[l][0][:c])
                assert np.array_equal(o.kv(l, 1, c), ar_kv[l][1][:c])
    assert rejects > 5


def test_external_rollback_truncates_and_reseeds():
    truth = ar_tokens("tiny", G)
    o = new_oracle(2)
    o.prefill(PROMPT)
    o.generate_spd(20, _draft_fn("right", truth, TINY.vocab, None))
    c = o.committed_len
    assert o.rollback(c + 1, 0) != 0 and o.rollback(-1, 0) != 0 and o.rollback(c, TINY.vocab) != 0
    new_c = c - 5
    assert o.rollback(new_c, truth[new_c - P]) == 0
    assert np.all(o.kv_len() == new_c) and o.fill == 1 and o.committed_len == new_c
    toks, _ = o.generate_spd(o.emitted + 10, _draft_fn("right", truth, TINY.vocab, None))
    assert toks[-10:] == list(truth[new_c - P + 1:new_c - P + 11])


# ------------------------------------------------------------------ independence / staircase -------

@pytest.mark.parametrize("n", [2, 4])
def test_in_flight_tokens_are_independent_and_match_ar_depth_states(n):
    truth = ar_tokens("tiny", G + 16)
    per = TINY.n_layers // n
    # AR residual stream after every layer, for positions P .. P+G
    ar = new_oracle(n)
    ar.prefill(PROMPT)
    trace = ar.ar_set_trace(True)
    ar_state = {}
    for i in range(G):
        ar.ar_step()
        ar_state[P + i] = trace.copy()
    a, b = new_oracle(n), new_oracle(n)
    b.set_forward_order(True)                                    # newest-first in step 3
    a.prefill(PROMPT)
    b.prefill(PROMPT)
    rng_a, rng_b = np.random.default_rng(5), np.random.default_rng(5)
    fa, fb = _draft_fn("random", truth, TINY.vocab, rng_a), _draft_fn("random", truth, TINY.vocab, rng_b)
    while a.emitted < G // 2:
        ra, rb = a.step(fa(a)), b.step(fb(b))
        assert ra == rb
        assert a.fill == b.fill
        depths = []
        for i in range(a.fill):
            pa, ta, ka, ha = a.ring(i)
            pb, tb, kb, hb = b.ring(i)
            assert (pa, ta, ka) == (pb, tb, kb) and np.array_equal(ha, hb)
            depths.append(ka)
            # a CORRECT in-flight token at depth k carries AR's residual stream after layer k*L/n - 1
            if all(a.ring(j)[1] == truth[a.ring(j)[0] - P] for j in range(i + 1)):
                assert np.array_equal(ha, ar_state[pa][ka * per])
        assert depths == list(range(a.fill - 1, -1, -1))         # depth staircase
        assert [a.ring(i)[0] for i in range(a.fill)] == list(range(a.committed_len, a.committed_len + a.fill))
    assert np.array_equal(a.kv_len(), b.kv_len())


def test_fill_runs_1_to_n_after_reject_then_stays_saturated():
    n = 4
    truth = ar_tokens("tiny", G + 16)
    o = new_oracle(n)
    o.prefill(PROMPT)
    fills = []
    # right drafts except one wrong draft at step 9
    for step in range(1, 30):
        pos_new = o.ring(o.fill - 1)[0]
        t = truth[pos_new + 1 - P]
        r = o.step((t + 1) % TINY.vocab if step == 9 else t)
        fills.append(r.fill)
    assert fills[:4] == [1, 2, 3, 4] and fills[4:9] == [4] * 5   # warm-up then saturated (Eq. 5 -> Eq. 2)
    # the wrong token entered at step 9 -> it is judged when its predecessor exits, n-1 steps later
    k = fills.index(1, 4)
    assert k == 9 + n - 1 and fills[k:k + 4] == [1, 2, 3, 4] and set(fills[k + 4:]) == {4}


def test_alpha_matches_closed_form():
    """i.i.d. successor-correctness p: a reject costs n cycles, an accept 1, so alpha = 1/(p+(1-p)n)
    (derived from PAPER.md:131 + :145)."""
    n, p, gen = 4, 0.6, 1500
    shape = shape_of("tiny", n)
    truth = np.array(ar_tokens("tiny", gen + 16), dtype=np.int32)
    o = Oracle(shape, weights("tiny", n), max_seq=P + gen + 64)
    o.prefill(PROMPT)
    o.set_forced(truth, p, 11)
    toks, log = o.generate_spd(gen)
    assert toks == list(truth[1:gen])
    alpha = (o.emitted - 1) / len(log)
    assert abs(alpha - 1.0 / (p + (1 - p) * n)) < 0.03
    saturated_rejects = [r for r in log if r.exited and not r.accepted and r.fill == n]
    assert all(r.discarded == n - 1 for r in saturated_rejects)


# ------------------------------------------------------------------ PDM as a pure function ---------

@pytest.mark.parametrize("n", [2, 4])
def test_pdm_is_a_pure_function_of_the_pre_step_slots(n):
    """Draft-token parity vs the PAPER's PDM is unpinned (different network, BASELINE.json overrides);
    what is pinned: slot j = pre-step state of the token at depth j, committed
    positions contribute Hfin (Eq. 5), and x_hat = argmax(E.RMSNorm(W_p.concat))."""
    shape = shape_of("tiny", n)
    w = weights("tiny", n)
    truth = ar_tokens("tiny", G + 16)
    o = new_oracle(n)
    o.prefill(PROMPT)
    d = TINY.d_model
    E = si.bf16_bits_to_f32(w["embed"])
    for step in range(12):
        a = o.fill
        ring = [o.ring(i) for i in range(a)]
        p_new = ring[-1][0]
        hf = {q: o.hfin(q) for q in range(max(0, p_new - n), o.committed_len)}
        r = o.step(truth[p_new + 1 - P] if step % 5 else (truth[p_new + 1 - P] + 3) % TINY.vocab)
        feats = o.last("pdm_feat").reshape(n, d)
        for j in range(n):
            if j < a:
                assert np.array_equal(feats[j], ring[a - 1 - j][3])          # pre-step state, depth j
                if j == 0:
                    assert np.array_equal(feats[0], E[ring[-1][1]])          # g^0: the bare embedding
            else:
                assert np.array_equal(feats[j], hf[p_new - j])               # committed -> depth-n feature
        ref = pdm_ref(shape, w, feats)
        np.testing.assert_allclose(o.last("pdm_prenorm"), ref["u"], rtol=1e-5, atol=1e-7)
        got = o.last("pdm_logits")
        assert np.max(np.abs(got - ref["logits"])) / np.max(np.abs(ref["logits"])) < 1e-5
        assert int(np.argmax(ref["logits"])) == int(np.argmax(got))
    # unforced, un-overridden: the step reports the PDM's own argmax
    r = o.step(-1)
    assert r.draft_token == int(np.argmax(o.last("pdm_logits"))) and r.draft_forced == 0


def test_config_validation():
    w = weights("tiny")
    with pytest.raises(ValueError):
        Oracle(TINY.replace(n_stages=3), w)                      # L % n != 0 (C-2.7)
    with pytest.raises(ValueError):
        Oracle(TINY.replace(n_q_heads=3), w)


# ------------------------------------------------------------------ the tie-hint test hook (ora_step_follow) ----
# The GPU parity harness lets the oracle continue with the CUDA path's token when the two argmaxes differ by less
# than the measured logit difference (tests/_parity.py).  These pins fix the hook itself: an inverted comparison,
# a relative-vs-absolute band mix-up or a missing range check would make the GPU token-exactness checks vacuous.

def _twin(n=2):
    a, b = new_oracle(n), new_oracle(n)
    assert a.prefill(PROMPT) == b.prefill(PROMPT)
    return a, b


def _runner_up(logits):
    order = np.argsort(-logits.astype(np.float64), kind="stable")
    return int(order[0]), int(order[1]), float(logits[order[0]] - logits[order[1]])


def test_tie_hint_band_zero_or_no_hint_is_the_plain_step():
    a, b = _twin(2)
    for i in range(12):
        ra = a.step()
        top, second, _ = _runner_up(a.last("pdm_logits"))
        rb = b.step_follow(second, (top + 1) % TINY.vocab, 0.0)        # band 0: never adopted
        assert tuple(ra) == tuple(rb)
    assert b.ties() == (0, 0)
    rb = b.step_follow(-1, -1, 1e9)                                    # no hint: nothing to adopt at any band
    assert tuple(a.step()) == tuple(rb) and b.ties() == (0, 0)
    a.close(); b.close()


def test_tie_hint_pdm_adopted_only_inside_the_absolute_band():
    """The PDM argmax: a hint whose oracle logit is `gap` below the maximum is ignored at band < gap, adopted at
    band > gap (and only then counted); the adopted token is the one that enters the pipeline."""
    a, b = _twin(4)
    ra = a.step()                                                      # the twin shows what this cycle's logits are
    top, second, gap = _runner_up(a.last("pdm_logits"))
    assert ra.draft_token == top and gap > 0 and not ra.exited
    c = new_oracle(4); c.prefill(PROMPT)
    rc = c.step_follow(second, -1, 0.9 * gap)
    assert tuple(rc) == tuple(ra) and c.ties() == (0, 0)               # outside the band: ignored
    rb = b.step_follow(second, -1, 1.1 * gap)
    assert rb.draft_token == second and b.ties() == (0, 1)             # inside: adopted, counted as a PDM tie
    assert b.ring(b.fill - 1)[1] == second                             # ... and it is what entered stage 0
    # the band is ABSOLUTE: scaled by max|logit| it would be far wider / narrower than the gap
    _, mx = a.margin(1)
    assert not (0.9 < mx < 1.1), "choose a config whose logit scale is not ~1, so relative vs absolute differ"
    d = new_oracle(4); d.prefill(PROMPT)
    rd = d.step_follow(second, -1, 0.9 * gap / mx if mx > 1 else 0.9 * gap * mx)   # what a relative reading would pass
    assert (d.ties() == (0, 0)) == (rd.draft_token == top)
    a.close(); b.close(); c.close(); d.close()


def test_tie_hint_rejects_far_and_invalid_tokens():
    """A comparison with the wrong sign would adopt the WORST token; out-of-range ids must never be adopted."""
    a, b = _twin(2)
    ra = a.step()
    lg = a.last("pdm_logits")
    worst = int(np.argmin(lg))
    top, _, gap = _runner_up(lg)
    for hint in (worst, TINY.vocab, TINY.vocab + 7, -5):
        c = new_oracle(2); c.prefill(PROMPT)
        rc = c.step_follow(hint, -1, 2.0 * gap)
        assert tuple(rc) == tuple(ra) and c.ties() == (0, 0), hint
        c.close()
    a.close(); b.close()


def test_tie_hint_verify_adopted_token_is_emitted_and_judges_the_successor():
    """At an exit the verify hint, if adopted, is the emitted token y: the successor is accepted iff it equals
    the hint, a reject reseeds with the hint (PAPER.md:129-131 applied to the adopted argmax)."""
    n = 2
    a, b = _twin(n)
    while True:                                                        # advance both to the cycle before an exit
        if a.ring(0)[2] == n - 1:
            break
        a.step(); b.step()
    succ = a.ring(1)[1] if a.fill > 1 else None
    ra = a.step()
    assert ra.exited
    top, second, gap = _runner_up(a.last("exit_logits"))
    assert ra.emitted_token == top
    c = new_oracle(n); c.prefill(PROMPT)
    while c.steps < b.steps:
        c.step()
    rc = c.step_follow(-1, second, 0.5 * gap)
    assert tuple(rc) == tuple(ra) and c.ties() == (0, 0)               # outside the band
    rb = b.step_follow(-1, second, 1.5 * gap)
    assert b.ties() == (1, 0) and rb.emitted_token == second
    assert rb.accepted == int(succ == second)
    if not rb.accepted:
        assert b.fill == 1 and b.ring(0)[1] == second and np.all(b.kv_len() == b.committed_len)
    a.close(); b.close(); c.close()


def test_longer_prefill_restricted_to_a_prefix_is_the_shorter_prefill():
    """Causality, as used by tests/golden/fullsize_golden.py (one 4096-token prefill serves the 2048-token config):
    cache rows and final hidden states below P of a 2P-token prefill equal the P-token prefill's bitwise, and an
    oracle loaded with those rows (ora_load_kv + ora_assume_prefilled) decodes the same greedy tokens."""
    shape = shape_of("tiny")
    w = weights("tiny")
    long_prompt = si.make_prompt(shape, 1, 2 * P)
    assert np.array_equal(long_prompt[:P], PROMPT)
    a = Oracle(shape, w, max_seq=2 * P + 32)
    a.prefill(long_prompt, block=16)
    b = Oracle(shape, w, max_seq=P + 32)
    first = b.prefill(PROMPT, block=16)
    for l in range(shape.n_layers):
        for which in (0, 1):
            assert np.array_equal(a.kv(l, which, P), b.kv(l, which, P))
    for pos in (0, P // 2, P - 1):
        assert np.array_equal(a.hfin(pos), b.hfin(pos))
    c = Oracle(shape, w, max_seq=P + 32)
    for l in range(shape.n_layers):
        c.load_kv(l, a.kv(l, 0, P), a.kv(l, 1, P))
    c.assume_prefilled(P, first)
    assert [b.ar_step() for _ in range(12)] == [c.ar_step() for _ in range(12)]
    a.close(); b.close(); c.close()
