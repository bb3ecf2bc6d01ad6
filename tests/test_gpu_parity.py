"""GPU-vs-oracle parity of the whole SPD path (-m gpu), through the C ABI, for all engines
(0 = one kernel per op, 1 = the fused persistent kernel with one stage chain per CTA, 2 = the fused persistent kernel with
multiplexed stage chains — the library's default; (2, c) = engine 2 with SPD_OPT_CHAINS = c).

Token ids, accept bits, fills, committed lengths and KV lengths: exact (ties within the logit tolerance
follow tests/_parity.py's protocol and are counted).  Hidden states, PDM vector and logits: max relative
error (C-2.18) within the north_star contract 2e-2, and within the tighter per-config bound DESIGN.md
derives from fp32 accumulation (1e-3 tiny, 1e-2 at the 4B/9B-class shapes).
"""
import numpy as np
import pytest

import spd_inputs as si
from tests._parity import run_parity, assert_ties, CONTRACT
from tests._util import TINY, shape_of, cached_last

pytestmark = pytest.mark.gpu

ENGINES = [0, 1, 2]
_HAS_MEGA = {}


def _need_engine(engine):
    e = engine[0] if isinstance(engine, tuple) else engine
    if e == 0:
        return
    if e not in _HAS_MEGA:
        import paper_2605_30852_b200 as spd
        g = spd.SPD(TINY, spd.upload_weights(si.make_weights(TINY)))
        try:
            g.set_option(spd.OPT.ENGINE, e)
            _HAS_MEGA[e] = True
        except spd.SpdError:
            _HAS_MEGA[e] = False
        finally:
            g.close()
    assert _HAS_MEGA[e], f"fused engine {e} must be available on a B200 (spd_create could not set it up)"


def _inputs(shape, prompt_len, seed=1234, std=0.02, random_gains=False, attention_heavy=False):
    import paper_2605_30852_b200 as spd

    def make():
        w = si.make_weights(shape, seed=seed, std=std, random_gains=random_gains, attention_heavy=attention_heavy)
        return dict(shape=shape, weights_np=w, dev_weights=spd.upload_weights(w), prompt=si.make_prompt(shape, seed, prompt_len))
    return dict(cached_last("parity_inputs", (shape, prompt_len, seed, std, random_gains, attention_heavy), make))   # a shallow copy: callers may replace entries


def _truth(shape, inp, n, block=16):
    from oracle import Oracle

    def make():
        o = Oracle(shape, inp["weights_np"], max_seq=len(inp["prompt"]) + n + 8)
        t = [o.prefill(inp["prompt"], block=block)] + [o.ar_step() for _ in range(n)]
        o.close()
        return np.array(t, np.int32)
    return cached_last("parity_truth", (id(inp["weights_np"]), shape, len(inp["prompt"]), n, block), make)


@pytest.mark.parametrize("engine", ENGINES)
def test_tiny_baseline_config_pdm_drafts(engine):
    """BASELINE.json configs[0] exactly: d256 L8 n2, std 0.02, gains 1, prompt 32, 64 greedy tokens,
    the PDM's own drafts."""
    _need_engine(engine)
    rep = run_parity(**_inputs(TINY, TINY.prompt_len), n_tokens=TINY.gen_len, engine=engine, tensor_tol=1e-3)
    print("tiny baseline:", rep.summary())
    assert rep.status == "ok", rep.detail
    assert_ties(rep)
    assert rep.emitted == TINY.gen_len - 1 and rep.verify_ties + rep.pdm_ties == 0


@pytest.mark.parametrize("engine", ENGINES)
@pytest.mark.parametrize("n", [1, 2, 4, 8])
@pytest.mark.parametrize("p", [0.0, 0.6, 1.0])
def test_tiny_hot_forced_acceptance(engine, n, p):
    """Diverse tokens (test-only init std 0.08, random gains), every pipeline width, accept/reject mixes."""
    _need_engine(engine)
    shape = shape_of("tiny", n)
    G = 40
    inp = _inputs(shape, 32, std=0.08, random_gains=True)
    rep = run_parity(**inp, n_tokens=G, forced=(_truth(shape, inp, G + 8), p, 7), engine=engine, tensor_tol=5e-3)
    print(f"tiny hot n={n} p={p}:", rep.summary())
    assert rep.status == "ok", rep.detail
    assert_ties(rep)
    if p == 1.0:
        assert rep.rejects == 0 and rep.steps == G + n - 2
    if p == 0.0 and n > 1:
        assert rep.rejects > 0


@pytest.mark.parametrize("engine", ENGINES)
def test_tiny_attention_heavy(engine):
    """W_o, W_v x8 and W_d /8 make attention errors visible in the hidden state (C-4)."""
    _need_engine(engine)
    rep = run_parity(**_inputs(TINY, 32, std=0.04, attention_heavy=True), n_tokens=48, engine=engine, tensor_tol=5e-3)
    print("attention heavy:", rep.summary())
    assert rep.status == "ok", rep.detail
    assert_ties(rep)


@pytest.mark.parametrize("engine", ENGINES)
@pytest.mark.parametrize("name,prompt_len,gen", [("4b_n4", 40, 20), ("4b_n8", 24, 14), ("9b_n4", 24, 12), ("9b_n16", 20, 10)])
def test_full_model_dims_short_prompt(engine, name, prompt_len, gen):
    """The 4B/9B-class shapes of BASELINE.json at every n, with a prompt short enough for the oracle:
    spans all tile shapes of the big configs (d 2560/4096, F 9728/12288, V 151936, ragged fills)."""
    _need_engine(engine)
    if engine == 1 and name not in ("4b_n4", "9b_n16"):
        pytest.skip("engine 1 (selectable, no longer the default) is checked at two of the four full-size shapes")
    shape = si.CONFIGS[name]
    inp = _inputs(shape, prompt_len)
    rep = run_parity(**inp, n_tokens=gen, forced=(_truth(shape, inp, gen + 2), 0.7, 3), engine=engine,
                     tensor_tol=1e-2, tensor_every=3)
    print(name, rep.summary())
    assert rep.status == "ok", rep.detail
    assert_ties(rep)
    assert rep.max_hidden_err < CONTRACT and rep.max_logit_err < CONTRACT


@pytest.mark.parametrize("engine", [1, 2])
@pytest.mark.parametrize("hq,hkv", [(8, 2), (8, 1), (4, 2), (2, 2)])
def test_tensor_core_attention_path_midsize(hq, hkv, engine):
    """head_dim 128 with a 300-token prompt: two full 128-row splits per head go through the fused engine's
    mma.sync attention (swizzled K/V boxes, q and probabilities split into bf16 hi + lo), the ragged third
    split through the scalar path; G = 4, 8 (q read from global), 2, 1.  Attention-heavy weights (C-4) make an
    attention error visible in the hidden state; compared with the oracle cycle by cycle at 5e-4."""
    _need_engine(engine)
    if engine == 2 and hq // hkv > 4:
        pytest.skip("engine 2 takes G <= 4 (spd_create falls back to engine 1 for this shape)")
    shape = si.ModelShape("mid", 512, 4, 2, hq, hkv, 128, 1024, 2048, 300, 24, ())
    inp = _inputs(shape, 300, std=0.04, attention_heavy=True)
    rep = run_parity(**inp, n_tokens=24, engine=engine, tensor_tol=5e-4, prefill_mode=0)   # the decode kernel's attention, prompt included
    print(f"mid Hq={hq} Hkv={hkv}:", rep.summary())
    assert rep.status == "ok", rep.detail
    assert_ties(rep)
    assert rep.max_hidden_err < 5e-4 and rep.max_logit_err < 5e-4


@pytest.mark.parametrize("chains", [1, 3, 4])
@pytest.mark.parametrize("n,p", [(4, 0.6), (8, 0.8), (8, None)])
def test_tiny_engine2_chain_counts(n, p, chains):
    """Engine 2 with 1, 3 and 4 stage chains per CTA (the default is 2): odd splits of the active stages into CTA groups
    (3 + 3 + 2 at n = 8, a single chain, bubbles after rejects) — results do not depend on the grouping."""
    _need_engine(2)
    shape = shape_of("tiny", n)
    inp = _inputs(shape, 32)
    G = 40
    forced = None if p is None else (_truth(shape, inp, G + 8), p, 7)
    rep = run_parity(**inp, n_tokens=G, forced=forced, engine=(2, chains), tensor_tol=5e-3)
    print(f"tiny n={n} p={p} chains={chains}:", rep.summary())
    assert rep.status == "ok", rep.detail
    assert_ties(rep)


@pytest.mark.parametrize("engine", [2, (2, 3)])
@pytest.mark.parametrize("n,p", [(4, 0.5), (8, 0.9)])
def test_tiny_long_generation_with_rejects(engine, n, p):
    """600 tokens (1000-2700 cycles, hundreds of rejects and refills, the context growing over five attention splits) cycle by
    cycle against the oracle: a soak of engine 2's stager / publisher / ring hand-overs at every fill level."""
    _need_engine(engine)
    shape = shape_of("tiny", n)
    inp = _inputs(shape, 32, seed=77)
    G = 600
    rep = run_parity(**inp, n_tokens=G, forced=(_truth(shape, inp, G + 16), p, 5), engine=engine, tensor_tol=5e-3,
                     tensor_every=16, max_seq=32 + 2 * G + 64)
    print(f"tiny long n={n} p={p} engine={engine}:", rep.summary())
    assert rep.status == "ok", rep.detail
    assert_ties(rep)
    assert rep.rejects > 20
