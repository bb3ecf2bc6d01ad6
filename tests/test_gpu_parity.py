"""GPU-vs-oracle parity of the whole SPD path (-m gpu), through the C ABI.

Token ids, accept bits, fills, committed lengths and KV lengths: exact.  Hidden states, PDM vector and
logits: max relative error (C-2.18) within the north_star contract 2e-2 — and, at the BASELINE init,
within the much tighter bound the arithmetic allows (fp32 re-association only, ~1e-5).
"""
import numpy as np
import pytest

import spd_inputs as si
from tests._parity import run_parity, run_parity_retry, CONTRACT
from tests._util import TINY, shape_of

pytestmark = pytest.mark.gpu

ENGINES = [0, 1]


def _engines_available():
    return ENGINES


def _inputs(shape, prompt_len, std=0.02, random_gains=False, attention_heavy=False):
    def make(seed):
        import paper_2605_30852_b200 as spd
        w = si.make_weights(shape, seed=seed, std=std, random_gains=random_gains, attention_heavy=attention_heavy)
        return dict(shape=shape, weights_np=w, dev_weights=spd.upload_weights(w),
                    prompt=si.make_prompt(shape, seed, prompt_len))
    return make


def _skip_if_engine_missing(engine):
    import paper_2605_30852_b200 as spd
    if engine == 1:
        shape = TINY
        w = spd.upload_weights(si.make_weights(shape))
        g = spd.SPD(shape, w)
        try:
            g.set_option(spd.OPT.ENGINE, 1)
        except spd.SpdError:
            pytest.skip("fused engine not built")
        finally:
            g.close()


@pytest.mark.parametrize("engine", ENGINES)
def test_tiny_baseline_config_pdm_drafts(engine):
    """BASELINE.json configs[0] exactly: d256 L8 n2, std 0.02, gains 1, prompt 32, 64 greedy tokens,
    the PDM's own drafts."""
    _skip_if_engine_missing(engine)
    rep = run_parity_retry(_inputs(TINY, TINY.prompt_len), seeds=[1234, 1235, 1236], n_tokens=TINY.gen_len,
                           engine=engine, tensor_tol=1e-3)
    assert rep.status == "ok", rep.detail
    assert rep.emitted == TINY.gen_len - 1
    print("tiny baseline", rep)


@pytest.mark.parametrize("engine", ENGINES)
@pytest.mark.parametrize("n", [1, 2, 4, 8])
@pytest.mark.parametrize("p", [0.0, 0.6, 1.0])
def test_tiny_hot_forced_acceptance(engine, n, p):
    """Diverse tokens (test-only init std 0.08, random gains), every pipeline width, accept/reject mixes."""
    _skip_if_engine_missing(engine)
    from tests._util import ar_tokens
    shape = shape_of("tiny", n)
    G = 40

    def make(seed):
        d = _inputs(shape, 32, std=0.08, random_gains=True)(seed)
        from oracle import Oracle
        o = Oracle(shape, d["weights_np"], max_seq=512)
        truth = [o.prefill(d["prompt"])] + [o.ar_step() for _ in range(G + 8)]
        o.close()
        d["forced"] = (np.array(truth, np.int32), p, 7)
        return d
    rep = run_parity_retry(make, seeds=[1234, 1235, 1236], n_tokens=G, engine=engine, tensor_tol=CONTRACT)
    assert rep.status == "ok", rep.detail
    if p == 1.0:
        assert rep.rejects == 0 and rep.steps == G + n - 2
    if p == 0.0 and n > 1:
        assert rep.rejects > 0
    print(f"tiny hot n={n} p={p}", rep.steps, rep.max_hidden_err, rep.max_logit_err, rep.detail)


@pytest.mark.parametrize("engine", ENGINES)
def test_tiny_attention_heavy(engine):
    """W_o, W_v x8 and W_d /8 make attention errors visible in the hidden state (C-4)."""
    _skip_if_engine_missing(engine)
    rep = run_parity_retry(_inputs(TINY, 32, std=0.04, attention_heavy=True), seeds=[1234, 1235, 1236],
                           n_tokens=48, engine=engine, tensor_tol=CONTRACT)
    assert rep.status == "ok", rep.detail
    print("attention heavy", rep.max_hidden_err, rep.max_logit_err)


@pytest.mark.parametrize("engine", ENGINES)
@pytest.mark.parametrize("name,prompt_len,gen", [("4b_n4", 40, 20), ("4b_n8", 24, 14), ("9b_n4", 24, 12), ("9b_n16", 20, 10)])
def test_full_model_dims_short_prompt(engine, name, prompt_len, gen):
    """The 4B/9B-class shapes of BASELINE.json at every n, with a prompt short enough for the oracle:
    spans all tile shapes of the big configs (d 2560/4096, F 9728/12288, V 151936)."""
    _skip_if_engine_missing(engine)
    shape = si.CONFIGS[name]
    from oracle import Oracle

    def make(seed):
        d = _inputs(shape, prompt_len)(seed)
        o = Oracle(shape, d["weights_np"], max_seq=prompt_len + gen + 8)
        truth = [o.prefill(d["prompt"], block=16)] + [o.ar_step() for _ in range(gen + 2)]
        o.close()
        d["forced"] = (np.array(truth, np.int32), 0.7, 3)
        return d
    rep = run_parity_retry(make, seeds=[1234, 1235], n_tokens=gen, engine=engine, tensor_tol=1e-3, tensor_every=3)
    assert rep.status == "ok", rep.detail
    print(name, rep.steps, rep.accepts, rep.rejects, rep.max_hidden_err, rep.max_logit_err, rep.min_margin, rep.detail)
