"""Pins for the oracle's paper-faithful Pipeline Draft Module.  CPU only.

What fixes the oracle here is not the oracle: a separately written float64 whole-prefix numpy model of the PDM
(oracle/nocache_ref.pdm_paper_ref: no KV cache, no cycle loop, library matmul — the whole feature sequence G_t is
rebuilt from the whole-prefix target forward every time), Eq. 3 by brute force from its definition, the paper's printed
anchor list for L = 32, the depth staircases of Eq. 2 / Eq. 5, the (n + 1)-row refresh of App. A.1
(PAPER.md:299), and the fact that verification does not depend on the drafter ("lossless").
"""
import numpy as np
import pytest

import spd_inputs as si
from oracle import Oracle
from oracle.nocache_ref import pdm_paper_ref
from tests._util import TINY, ar_tokens, shape_of, weights

P = TINY.prompt_len
PROMPT = si.make_prompt(TINY, 1)
HOT = dict(std=0.08, random_gains=True)


def pdm_oracle(n, pdm_layers=2, pdm_vocab=300, max_seq=512, **wkw):
    shape = shape_of("tiny", n)
    kw = dict(HOT, **wkw)
    w = weights("tiny", n, **kw)
    pw = si.make_pdm_weights(shape, pdm_layers, pdm_vocab, seed=1234, std=kw["std"], random_gains=kw["random_gains"])
    o = Oracle(shape, w, max_seq=max_seq)
    o.attach_pdm(pw)
    return shape, w, pw, o


def test_anchor_set_is_the_papers_for_32_layers_and_f_is_eq3():
    """PAPER.md:91 / :295: for L = 32 the anchors are [0, 8, 16, 24, 31]; Eq. 3: f(k) = max{i | b_i <= min(L, k L/n)}."""
    for L, n in ((32, 4), (32, 8), (32, 16), (8, 2), (8, 4), (8, 8), (12, 3)):
        shape = TINY.replace(n_layers=L, n_stages=n)
        w = si.make_weights(shape.replace(n_layers=1), seed=1)          # only shapes matter here
        w = {k: (v * L if isinstance(v, list) else v) for k, v in w.items()}
        o = Oracle(shape, w, max_seq=8)
        B = o.pdm_anchors()
        if L == 32:
            assert B == [0, 8, 16, 24, 31]
        assert B[0] == 0 and B[-1] == L - 1 and B == sorted(set(B))
        for k in range(n + 1):
            lmax = min(L, k * L // n)
            assert o.pdm_f(k) == max(i for i, b in enumerate(B) if b <= lmax)
        assert o.pdm_f(0) == 0 and o.pdm_f(n) == len(B) - 1              # k = 0: the embedding only; k = n: every anchor
        o.close()


def test_anchors_are_the_targets_hidden_states_entering_the_anchor_layers():
    """H^b of a committed position = O-AR's residual stream after layer b - 1 (trace[b]); H^0 = the embedding."""
    shape, w, pw, o = pdm_oracle(2)
    ref = Oracle(shape, w, max_seq=512)
    ref.prefill(PROMPT)
    tr = ref.ar_set_trace(True)
    o.prefill(PROMPT)
    B = o.pdm_anchors()
    truth = ar_tokens("tiny", 12)
    for i in range(6):
        pos = P + i
        ref.ar_step()
        # drive o with the right drafts so position pos gets committed with the same token sequence
        while o.committed_len <= pos:
            o.step(truth[o.ring(o.fill - 1)[0] + 1 - P])
        for j, b in enumerate(B):
            assert np.array_equal(o.pdm_anchor(pos, j), tr[b]), (pos, b)
    o.close(); ref.close()


BASE = dict(std=0.02, random_gains=False)     # BASELINE.json's init: the two models agree to ~1e-5 (no chaotic K/V rounding flips)


@pytest.mark.parametrize("n,pdm_layers,mode,init,tol", [
    (2, 2, "pdm", BASE, 2e-4), (4, 1, "forced", BASE, 2e-4), (4, 3, "pdm", BASE, 2e-4), (1, 2, "pdm", BASE, 2e-4),
    (8, 2, "forced", BASE, 2e-4), (4, 2, "forced", HOT, 2e-2), (2, 2, "pdm", HOT, 2e-2)])
def test_pdm_matches_the_whole_prefix_float64_model(n, pdm_layers, mode, init, tol):
    """Every cycle: logits, last hidden state, features and drafted token against the no-cache float64 model rebuilt
    from the whole token sequence (verified prefix + in-flight tokens) with the depths the ring holds before the step."""
    shape, w, pw, o = pdm_oracle(n, pdm_layers, **init)
    first = o.prefill(PROMPT)
    committed = list(PROMPT)
    truth = ar_tokens("tiny", 40, std=init["std"], random_gains=init["random_gains"])
    if mode == "forced":
        o.set_forced(np.array(truth, np.int32), 0.7, 11)
    exits = rejects = 0
    for cyc in range(14 if n <= 4 else 20):
        ring = [o.ring(i) for i in range(o.fill)]
        c = o.committed_len
        assert [r[0] for r in ring] == list(range(c, c + len(ring)))
        tokens = committed + [r[1] for r in ring]
        depths = [n] * c + [r[2] for r in ring]                 # Eq. 2 / Eq. 5: prefix at depth n, then the staircase
        assert [r[2] for r in ring] == list(range(len(ring) - 1, -1, -1))
        res = o.step()
        first_row, row_depths = o.pdm_rows()
        assert list(row_depths) == depths[first_row:]
        assert len(row_depths) <= n + 1 or cyc == 0             # only the trailing n+1 features are refreshed
        ref = pdm_paper_ref(shape, w, pw, tokens, depths)
        lg = o.pdm_last("logits")
        scale = np.abs(ref["logits"]).max()
        assert np.abs(lg - ref["logits"]).max() <= tol * scale, cyc
        np.testing.assert_allclose(o.pdm_last("features"), ref["features"][first_row:], atol=tol * np.abs(ref["features"]).max())
        assert np.abs(o.pdm_last("hidden") - ref["hidden"]).max() <= tol * np.abs(ref["hidden"]).max()
        gap = np.sort(ref["logits"])[-1] - np.sort(ref["logits"])[-2]
        if not res.draft_forced and gap > 2 * tol * scale:
            assert res.draft_token == ref["token"] and res.draft_token in set(pw["vocab_map"])
        # the PDM's cache after the run: rows of every layer equal the whole-prefix K/V (bf16, boundary flips aside)
        T = len(tokens)
        for l in (0, pdm_layers - 1):
            for which, name in ((0, "k"), (1, "v")):
                rows, fin = o.pdm_kv(l, which, T)
                assert fin == c
                got = si.bf16_bits_to_f32(rows).astype(np.float64)
                want = ref[name][l]
                assert np.all(np.abs(got - want) <= 2.0 ** -7 * np.abs(want) + tol * np.abs(want).max())
        if res.exited:
            exits += 1
            rejects += 1 - res.accepted
            committed.append(ring[0][1])
    assert exits > 0 and (n == 1 or rejects > 0)
    o.close()


@pytest.mark.parametrize("n", [1, 2, 4])
def test_verification_is_lossless_with_the_papers_pdm(n):
    """whatever the drafter proposes, the emitted tokens are plain greedy decode."""
    shape, w, pw, o = pdm_oracle(n, 2)
    first = o.prefill(PROMPT)
    toks, log = o.generate_spd(24)
    assert [first] + toks == list(ar_tokens("tiny", 24))
    assert all(r.discarded == r.fill - 1 for r in log if r.exited and not r.accepted)
    o.close()


def test_full_depth_rows_are_final_and_rollback_rewinds_them():
    """A committed position's PDM rows do not change once built at depth n (they "remain valid across steps and may be
    KV-cached"); an external rollback into the committed prefix rebuilds the rows above it."""
    shape, w, pw, o = pdm_oracle(4, 2)
    o.prefill(PROMPT)
    o.step()
    k0, fin = o.pdm_kv(1, 0, P)
    assert fin == P
    for _ in range(9):
        o.step()
    k1, fin1 = o.pdm_kv(1, 0, P)
    assert np.array_equal(k0, k1) and fin1 == o.committed_len or fin1 <= o.committed_len
    c = o.committed_len
    assert o.rollback(c - 2, 5) == 0
    o.step()
    first_row, depths = o.pdm_rows()
    assert first_row == c - 2 and list(depths) == [0]          # position c-2 is the reseed token (depth 0); below: final
    o.close()


def test_attach_validation_and_greedy_only():
    shape = shape_of("tiny", 2)
    w = weights("tiny", 2)
    pw = si.make_pdm_weights(shape, 1, 64, seed=3)
    o = Oracle(shape, w, max_seq=64)
    bad = dict(pw); bad["vocab_map"] = pw["vocab_map"][::-1].copy()
    with pytest.raises(ValueError):
        o.attach_pdm(bad)                                       # the map must be strictly ascending
    bad = dict(pw); bad["vocab"] = shape.vocab + 1
    with pytest.raises(ValueError):
        o.attach_pdm(bad)
    o.attach_pdm(pw)
    with pytest.raises(ValueError):
        o.set_sampling(1.0, 50, 1)                              # reading P-9: sampling with the paper's PDM is not built
    o.close()
