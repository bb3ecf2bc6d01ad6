"""Writes tests/golden/fullsize_<config>.npz: what the ORACLE computes at BASELINE.json's full prompt lengths.

Calls only oracle/ and spd_inputs/ (never the CUDA path).  Why stored values: the oracle's 2048-token prefill of the
9B-class model is ~14 T fp64 multiply-adds (about 10 minutes on 16 host cores, 20 for the 4096-token prompt) and the
driver gives the whole `pytest -m gpu` run 20 minutes, so the full-size oracle tier ("prefill result +
the first 32 emitted tokens + spot-checked slot states") compares the CUDA path with the values this script stored.
`SPD_FULL_TIER=live` makes tests/test_gpu_fullsize.py call compute() in-process instead of loading the files.

Everything stored is a quantity of plain greedy decode O-AR (every SPD run must reproduce it), keyed
by POSITION, so it is valid for any pipeline width n, any acceptance pattern and any cycle count:
  tokens[i]        the token at position P + i (tokens[0] = argmax of the last prompt position's logits)
  hfin[j]          final (pre-norm) hidden state of position hfin_pos0 + j  (Eq. 5 warm-up features and every exit)
  top_idx/top_val  the 32 largest logits of the vector that decides tokens[i] (the tie protocol needs the runner-ups)
  logit_idx/_val   2048 seeded sample entries of that vector (the measured logit difference)
  kv_pos/k_rows/v_rows   bf16 K and V rows of layers kv_layers at sampled prompt positions
  trace            O-AR's residual stream after layer b - 1 for b in trace_layers at positions trace_pos: the state an
                   in-flight token must hold after completing b / (L/n) stages (SURVEY C-3 "in-flight hidden states")

    python tests/golden/fullsize_golden.py 9b      # 9b_n4 (P = 2048) and 9b_n16 (P = 4096) from ONE 4096-token prefill
    python tests/golden/fullsize_golden.py 4b_n8   # P = 1024
"""
from __future__ import annotations

import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle as ora  # noqa: E402
import spd_inputs as si  # noqa: E402

SEED = 1234
GEN = {"9b_n4": 32, "9b_n16": 8, "4b_n8": 32}        # emitted tokens compared at full size (SURVEY C-4 tiers)
HFIN_BACK = 16                                        # prompt positions P-16 .. P-1 (PDM warm-up slots, n <= 16)
N_SAMPLE, N_TOP = 2048, 32


def path(name: str) -> str:
    return os.path.join(HERE, f"fullsize_{name}.npz")


def load(name: str) -> dict:
    with np.load(path(name)) as z:
        return {k: z[k] for k in z.files}


def trace_layers(shape) -> np.ndarray:
    """Stage boundaries b = k * L/n kept in the golden (at most four depths k)."""
    n, per = shape.n_stages, shape.n_layers // shape.n_stages
    ks = sorted({1, max(1, n // 3), max(1, (2 * n) // 3), n - 1}) if n > 1 else []
    return np.array([k * per for k in ks], dtype=np.int32)


def _head(shape, w, h):
    """logits = E . RMSNorm(h; g_final) from the oracle's single operations (C-1)."""
    return ora.op_gemv(w["embed"], ora.op_rmsnorm(h, w["final_norm"], shape.rms_eps))


def _kv_positions(P: int) -> np.ndarray:
    cand = [0, 1, 2, 63, 127, 128, 129, 255, 256, P // 4, P // 2 - 1, P // 2, P // 2 + 1, (3 * P) // 4, P - 130, P - 129,
            P - 128, P - 3, P - 2, P - 1]
    return np.array(sorted({p for p in cand if 0 <= p < P}), dtype=np.int32)


def _collect(shape, w, o, P: int, G: int, first_logits: np.ndarray, hfin_prompt: np.ndarray, log=print) -> dict:
    """`o` is an oracle whose committed length is P with the first token pending; runs G greedy steps."""
    rng = np.random.Generator(np.random.PCG64([SEED, 4242]))
    sample = np.sort(rng.choice(shape.vocab, size=min(N_SAMPLE, shape.vocab), replace=False)).astype(np.int32)
    tl = trace_layers(shape)
    kv_layers = np.array(sorted({0, shape.n_layers // 2 - 1, shape.n_layers - 1}), dtype=np.int32)
    kv_pos = _kv_positions(P)
    g = {"prompt_len": np.int32(P), "seed": np.int32(SEED), "hfin_pos0": np.int32(P - HFIN_BACK), "logit_idx": sample,
         "trace_layers": tl, "kv_layers": kv_layers, "kv_pos": kv_pos}
    g["k_rows"] = np.stack([o.kv(int(l), 0, P)[kv_pos] for l in kv_layers])
    g["v_rows"] = np.stack([o.kv(int(l), 1, P)[kv_pos] for l in kv_layers])
    tokens, top_idx, top_val, lval, maxabs, hf, trace, trace_pos = [], [], [], [], [], [hfin_prompt], [], []

    def keep(logits):
        order = np.argsort(-logits.astype(np.float64), kind="stable")[:N_TOP]
        tokens.append(int(order[0]))
        top_idx.append(order.astype(np.int32)); top_val.append(logits[order]); lval.append(logits[sample])
        maxabs.append(float(np.max(np.abs(logits))))

    keep(first_logits)
    tr = o.ar_set_trace(True)
    every = 4 if G >= 16 else 2
    for i in range(G):
        t0 = time.time()
        pos = P + i
        y = o.ar_step()
        lg = o.last("exit_logits")
        keep(lg)
        assert tokens[-1] == y
        hf.append(o.hfin(pos)[None, :])
        if i % every == 0 and len(tl):
            trace.append(tr[tl].copy()); trace_pos.append(pos)
        log(f"  AR step {i + 1}/{G}: position {pos} -> token {y} ({time.time() - t0:.1f} s)")
    o.ar_set_trace(False)
    g.update(tokens=np.array(tokens, np.int32), top_idx=np.stack(top_idx), top_val=np.stack(top_val).astype(np.float32),
             logit_val=np.stack(lval).astype(np.float32), logit_maxabs=np.array(maxabs, np.float32),
             hfin=np.concatenate(hf).astype(np.float32),
             trace=np.stack(trace).astype(np.float32) if trace else np.zeros((0, 0, shape.d_model), np.float32),
             trace_pos=np.array(trace_pos, np.int32))
    return g


def compute(name: str, block: int = 16, log=print) -> dict:
    """One config from its own full-length oracle prefill."""
    shape = si.CONFIGS[name]
    P, G = shape.prompt_len, GEN[name]
    w = si.make_weights(shape, seed=SEED)
    prompt = si.make_prompt(shape, SEED)
    o = ora.Oracle(shape, w, max_seq=P + G + 8)
    t0 = time.time()
    first = o.prefill(prompt, block=block)
    log(f"{name}: oracle prefill of {P} tokens (block {block}) took {time.time() - t0:.0f} s on {ora.num_threads()} threads")
    lg = o.last("exit_logits")
    assert int(np.argmax(lg)) == first
    hfp = np.stack([o.hfin(p) for p in range(P - HFIN_BACK, P)])
    g = _collect(shape, w, o, P, G, lg, hfp, log)
    o.close()
    return g


def compute_9b_pair(block: int = 16, log=print) -> dict:
    """9b_n4 (prompt 2048) and 9b_n16 (prompt 4096) share the decoder weights (the generator keys a tensor on (seed,
    name, layer); only W_p depends on n, and O-AR never reads it) and 9b_n4's prompt is the first half of 9b_n16's, so
    ONE 4096-token prefill serves both: by causality its cache rows and hidden states below 2048 are those of the
    2048-token prefill (the blocked prefill treats every token exactly as the plain one does)."""
    s4, s16 = si.CONFIGS["9b_n4"], si.CONFIGS["9b_n16"]
    w = si.make_weights(s16, seed=SEED)
    p16, p4 = si.make_prompt(s16, SEED), si.make_prompt(s4, SEED)
    assert np.array_equal(p16[:len(p4)], p4)
    for key, layer in (("wq", 0), ("w_down", s4.n_layers - 1), ("final_norm", -1)):
        t = si.make_tensor(s4, key, layer, SEED)
        assert np.array_equal(t, w[key][layer] if layer >= 0 else w[key])
    P16, P4 = len(p16), len(p4)
    o = ora.Oracle(s16, w, max_seq=P16 + GEN["9b_n16"] + 8)
    t0 = time.time()
    first16 = o.prefill(p16, block=block)
    log(f"9b: oracle prefill of {P16} tokens (block {block}) took {time.time() - t0:.0f} s on {ora.num_threads()} threads")
    # the state at P = 2048, before the longer run moves on
    o4 = ora.Oracle(s4, w, max_seq=P4 + GEN["9b_n4"] + 8)
    for l in range(s4.n_layers):
        o4.load_kv(l, o.kv(l, 0, P4), o.kv(l, 1, P4))
    hfp4 = np.stack([o.hfin(p) for p in range(P4 - HFIN_BACK, P4)])
    lg4 = _head(s4, w, o.hfin(P4 - 1))
    o4.assume_prefilled(P4, int(np.argmax(lg4)))
    lg16 = o.last("exit_logits")
    assert int(np.argmax(lg16)) == first16
    hfp16 = np.stack([o.hfin(p) for p in range(P16 - HFIN_BACK, P16)])
    out = {"9b_n16": _collect(s16, w, o, P16, GEN["9b_n16"], lg16, hfp16, log)}
    o.close()
    out["9b_n4"] = _collect(s4, w, o4, P4, GEN["9b_n4"], lg4, hfp4, log)
    o4.close()
    return out


def main(argv):
    what = argv[1] if len(argv) > 1 else "9b"
    if what == "9b":
        for name, g in compute_9b_pair().items():
            np.savez(path(name), **g)
            print("wrote", path(name), os.path.getsize(path(name)), "bytes")
    else:
        g = compute(what)
        np.savez(path(what), **g)
        print("wrote", path(what), os.path.getsize(path(what)), "bytes")


if __name__ == "__main__":
    main(sys.argv)
