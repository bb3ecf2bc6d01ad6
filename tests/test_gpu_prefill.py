"""The batched tensor-core prefill (prefill is the step before the timed path)
against the oracle (-m gpu), through the C ABI.

  * spd_op_gemm — the tcgen05 GEMM alone (fp32 activations as three bf16 parts (exact), exact bf16 weights, fp32 accumulation in
    TMEM) against the oracle's GEMV row by row: full tiles, ragged M / N tails, K from 64 to 12288;
  * spd_prefill with SPD_OPT_PREFILL = 1 against the oracle's prefill: first token, final hidden states of every
    position, K/V rows of every layer (one bf16 ulp + tolerance), and then the decode cycles that start from that
    state (run_parity: tokens exact, tensors within tolerance);
  * against SPD_OPT_PREFILL = 0 (the prompt through the decode kernel): same first token, K/V rows within one bf16 ulp.
"""
import numpy as np
import pytest
import torch

import oracle as ora
import spd_inputs as si
from tests._parity import run_parity, assert_ties, rel_err
from tests._util import TINY, shape_of

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("M,N,K", [(128, 256, 64), (1, 8, 64), (300, 1000, 256), (129, 260, 4096), (64, 704, 12288),
                                   (1024, 512, 1024)])
def test_op_gemm_matches_the_oracle_gemv(M, N, K):
    import paper_2605_30852_b200 as spd
    rng = np.random.default_rng(M * 7 + N)
    x = (rng.standard_normal((M, K)) * 1.7).astype(np.float32)
    w = si.f32_to_bf16_bits((rng.standard_normal((N, K)) * 0.05).astype(np.float32))
    y = spd.op_gemm(torch.from_numpy(x).cuda(), torch.from_numpy(w.view(np.int16)).cuda()).cpu().numpy()
    rows = sorted(set([0, M // 2, M - 1] + list(rng.integers(0, M, 5))))
    for m in rows:
        want = ora.op_gemv(w, x[m])
        e = rel_err(y[m], want)
        assert e < 1e-4, f"row {m}: rel err {e:.2e}"      # SURVEY C-4: per-kernel parity <= 1e-4
    # all rows against float64 matmul of the same operands (the oracle's definition, as a library routine)
    ref = x.astype(np.float64) @ si.bf16_bits_to_f32(w).astype(np.float64).T
    assert rel_err(y, ref) < 1e-4


def _kv_close(g_bits, o_bits, tol, what):
    g = si.bf16_bits_to_f32(g_bits).astype(np.float64)
    o = si.bf16_bits_to_f32(o_bits).astype(np.float64)
    lim = 2.0 ** -7 * np.abs(o) + tol * np.max(np.abs(o))
    assert np.all(np.abs(g - o) <= lim), what
    return float(np.mean(g != o))


@pytest.mark.parametrize("name,n,P,kw,tol", [
    ("tiny", 2, 32, dict(), 1e-3),
    ("tiny", 4, 150, dict(std=0.08, random_gains=True), 5e-3),            # ragged M tile, 3 attention tiles
    ("tiny", 2, 97, dict(std=0.04, attention_heavy=True), 5e-3),
    ("mid", 2, 300, dict(std=0.04, attention_heavy=True), 5e-4),          # head_dim 128, G = 4
    ("4b_n4", 4, 140, dict(), 1e-2),                                      # the 4B-class tile shapes (F = 9728)
])
def test_batched_prefill_against_the_oracle(name, n, P, kw, tol):
    import paper_2605_30852_b200 as spd
    shape = si.ModelShape("mid", 512, 4, 2, 8, 2, 128, 1024, 2048, P, 16, ()) if name == "mid" else shape_of(name, n)
    w = si.make_weights(shape, seed=1234, **kw)
    wd = spd.upload_weights(w)
    prompt = si.make_prompt(shape, 7, P)
    o = ora.Oracle(shape, w, max_seq=P + 8)
    fo = o.prefill(prompt, block=16)
    g = spd.SPD(shape, wd, max_seq=P + 64)
    g.set_option(spd.OPT.PREFILL, 1)
    g.set_option(spd.OPT.DEBUG_LOGITS, 1)
    fg = g.prefill(prompt)
    lg, lo = g.last("exit_logits"), o.last("exit_logits")
    assert rel_err(lg, lo) < tol and int(np.argmax(lg)) == fg
    gap, mx = o.margin(0)
    assert fg == fo or lo[fo] - lo[fg] <= 3.0 * float(np.max(np.abs(lg.astype(np.float64) - lo)))
    assert np.all(g.kv_len() == P)
    worst = max(rel_err(g.hfin(p), o.hfin(p)) for p in range(P))
    assert worst < tol, f"final hidden states: {worst:.2e}"
    flips = 0.0
    for l in range(shape.n_layers):
        for which in (0, 1):
            flips = max(flips, _kv_close(g.kv(l, which, P), o.kv(l, which, P), tol, f"layer {l} {'KV'[which]} rows"))
    # the other prefill path (the prompt through the decode kernel): same token, rows within one bf16 ulp
    h = spd.SPD(shape, wd, max_seq=P + 64)
    h.set_option(spd.OPT.PREFILL, 0)
    fh = h.prefill(prompt)
    worst_h = max(rel_err(h.hfin(p), o.hfin(p)) for p in range(P))
    assert fh == fg or fg != fo
    for l in (0, shape.n_layers - 1):
        for which in (0, 1):
            _kv_close(g.kv(l, which, P), h.kv(l, which, P), tol, f"layer {l}: batched vs pipelined prefill")
    print(f"{name} n={n} P={P}: first {fg}/{fo}/{fh} hfin {worst:.2e} (pipelined prefill: {worst_h:.2e}) logits {rel_err(lg, lo):.2e} kvflip {flips:.3f}")
    o.close(); g.close(); h.close()


@pytest.mark.parametrize("engine", [0, 1, 2])
def test_decode_after_batched_prefill_matches_the_oracle(engine):
    """run_parity uses the library's default prefill (the batched one): cycles that start from its state."""
    import paper_2605_30852_b200 as spd
    shape = shape_of("tiny", 4)
    w = si.make_weights(shape, seed=1234, std=0.08, random_gains=True)
    g = spd.SPD(shape, spd.upload_weights(w), max_seq=400)
    g.set_option(spd.OPT.PREFILL, 1)         # raises if the batched prefill is not available on this box
    g.close()
    rep = run_parity(shape=shape, weights_np=w, dev_weights=spd.upload_weights(w), prompt=si.make_prompt(shape, 1, 70),
                     n_tokens=30, engine=engine, tensor_tol=5e-3)
    print("decode after batched prefill:", rep.summary())
    assert rep.status == "ok", rep.detail
    assert_ties(rep)
