"""Differential test of the C ABI's state machine (-m gpu): seeded random sequences of calls — cycles in greedy,
forced-acceptance and sampling mode, external rollbacks, mode switches on a live pipeline, re-prefills — run on the
CUDA library and on the oracle side by side; after every call the step results, the ring (fill, committed length,
per-depth position and token), the per-layer KV lengths and the counters K, N must be identical.  The sequences
are fixed by their seed, both sides are deterministic, so is the test.  Decisions that floating point takes within
the measured logit difference of their boundary follow tests/_parity.py's protocols (the oracle is told what the
CUDA path decided and adopts it only then); the adoptions are counted and bounded."""
import numpy as np
import pytest

import spd_inputs as si
from oracle import Oracle
from tests._util import shape_of

pytestmark = pytest.mark.gpu


def _state_equal(gpu, ora, what):
    fill, c, slots = gpu.ring()
    assert (fill, c) == (ora.fill, ora.committed_len), what
    for i in range(ora.fill):
        pos, tok, k, _ = ora.ring(i)
        assert slots[k] == (1, pos, tok), f"{what}: depth {k}"
    assert np.array_equal(gpu.kv_len(), ora.kv_len()), what
    K, N, _ = gpu.counters()
    assert (K, N) == (ora.steps, ora.emitted), what


@pytest.mark.parametrize("engine", [0, 1, 2])
@pytest.mark.parametrize("n,seed", [(1, 0), (2, 1), (4, 2), (4, 3), (8, 4), (2, 5), (4, 6), (8, 7), (1, 8), (4, 9), (2, 10),
                                    (8, 11)])
def test_random_call_sequences_match_the_oracle(engine, n, seed):
    import paper_2605_30852_b200 as spd
    shape = shape_of("tiny", n, vocab=64)
    w = si.make_weights(shape, seed=1234, std=0.08, random_gains=True)
    rng = np.random.default_rng(1000 + seed)
    ms = 640
    gpu = spd.SPD(shape, spd.upload_weights(w), max_seq=ms)
    ora = Oracle(shape, w, max_seq=ms)
    log = []
    try:
        gpu.set_option(spd.OPT.ENGINE, engine)
        gpu.set_option(spd.OPT.DEBUG_LOGITS, 1)
        delta, ties = [0.0], [0, 0]      # largest logit difference measured so far; adoptions (sampling, argmax)

        def measure(what):
            d = float(np.max(np.abs(ora.last(what).astype(np.float64) - gpu.last(what))))
            assert d < 5e-3 * max(1.0, float(np.max(np.abs(ora.last(what))))), f"{log[-4:]}: {what} differ by {d:.2e}"
            delta[0] = max(delta[0], d)

        def prefill():
            P = int(rng.integers(1, 40))
            prompt = rng.integers(0, shape.vocab, P).astype(np.int32)
            fg, fo = gpu.prefill(prompt), ora.prefill(prompt, block=int(rng.integers(1, 9)))
            log.append(f"prefill({P})")
            measure("exit_logits")
            assert fg == fo, log[-1]
            return P

        mode = "greedy"
        P = prefill()
        for op_i in range(60):
            op = rng.choice(["steps", "steps", "steps", "rollback", "forced", "sampling", "greedy", "prefill"],
                            p=[0.3, 0.2, 0.1, 0.1, 0.1, 0.1, 0.05, 0.05])
            if ora.committed_len + 40 >= ms - 2 * n - 8:
                op = "prefill"
            if op == "steps":
                k = int(rng.integers(1, 13))
                many = bool(rng.integers(0, 2)) and mode != "sampling"   # sampling: the per-cycle record is needed
                log.append(f"steps({k}, many={many}, mode={mode})")
                if mode == "sampling":
                    for _ in range(k):
                        a = gpu.step()
                        rec = gpu.sample_record()
                        band = 3.0 * delta[0] + 1e-5
                        b = ora.step_sample_follow(draft_ids=rec["draft"][0], verify_ids=rec["target"][0] if a.exited else None,
                                                   draft_token=a.draft_token, accepted=a.accepted if a.exited else -1,
                                                   emitted_token=a.emitted_token if a.exited and not a.accepted else -1,
                                                   logit_band=band, prob_eps=4.0 * band)
                        assert tuple(a) == tuple(b), f"{log[-8:]}: gpu {tuple(a)} != oracle {tuple(b)} (band {band:.1e})"
                        measure("pdm_logits")
                        if a.exited:
                            measure("exit_logits")
                    ties[0] = sum(ora.sample_record()["ties"])
                else:
                    rg = gpu.step_many(k) if many else [gpu.step() for _ in range(k)]
                    for a in rg:
                        b = ora.step_follow(-1 if a.draft_forced else a.draft_token, a.emitted_token if a.exited else -1, 3.0 * delta[0] + 1e-5)
                        assert tuple(a) == tuple(b), f"{log[-8:]}: gpu {tuple(a)} != oracle {tuple(b)}"
                    ties[1] = sum(ora.ties())
            elif op == "rollback":
                new_len = int(rng.integers(max(1, ora.committed_len - 6), ora.committed_len + 1))
                tok = int(rng.integers(0, shape.vocab))
                log.append(f"rollback({new_len}, {tok})")
                gpu.rollback(new_len, tok)
                assert ora.rollback(new_len, tok) == 0
            elif op == "forced":
                if mode == "sampling":
                    gpu.set_sampling(1.0, 0, 0); ora.set_sampling(1.0, 0, 0)
                p = float(rng.choice([0.0, 0.3, 0.7, 1.0]))
                truth = rng.integers(0, shape.vocab, int(rng.integers(0, 200))).astype(np.int32)
                log.append(f"forced(p={p}, n_truth={len(truth)})")
                gpu.set_forced(truth, p, seed + op_i); ora.set_forced(truth, p, seed + op_i)
                mode = "forced"
            elif op == "sampling":
                gpu.set_forced(None, -1.0, 0); ora.set_forced(None, -1.0, 0)
                T, k = float(rng.choice([0.7, 1.0, 2.0])), int(rng.choice([1, 5, 50, 64]))
                log.append(f"sampling(T={T}, k={k})")
                gpu.set_sampling(T, k, 77 + op_i); ora.set_sampling(T, k, 77 + op_i)
                mode = "sampling"
            elif op == "greedy":
                log.append("greedy")
                gpu.set_forced(None, -1.0, 0); ora.set_forced(None, -1.0, 0)
                gpu.set_sampling(1.0, 0, 0); ora.set_sampling(1.0, 0, 0)
                mode = "greedy"
            else:
                P = prefill()
            _state_equal(gpu, ora, str(log[-8:]))
        assert sum(s.startswith("steps") for s in log) >= 15
        print(f"fuzz n={n} seed={seed} engine={engine}: {len(log)} calls, max logit diff {delta[0]:.2e}, "
              f"adoptions sampling/argmax {ties}")
        assert ties[0] + ties[1] <= 4
    finally:
        gpu.close()
        ora.close()
