"""Seeded generators: model shapes, bf16 weights, prompts.  No SPD arithmetic lives here."""
from __future__ import annotations

import ctypes
import dataclasses
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_FASTGEN = None


def _fastgen():
    """gcc-built helper (spd_inputs/fastgen.c): fills a bf16 matrix with seeded N(0, std) values."""
    global _FASTGEN
    if _FASTGEN is None:
        src = os.path.join(_HERE, "fastgen.c")
        lib = os.path.join(_HERE, "libfastgen.so")
        if not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(src):
            subprocess.run(["gcc", "-std=c11", "-O2", "-march=x86-64-v3", "-ffp-contract=off", "-fopenmp",
                            "-fPIC", "-shared", "-o", lib, src, "-lm"], check=True)
        L = ctypes.CDLL(lib)
        L.fastgen_normal_bf16.argtypes = [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_float]
        L.fastgen_normal_bf16.restype = None
        _FASTGEN = L
    return _FASTGEN


@dataclasses.dataclass(frozen=True)
class ModelShape:
    """One BASELINE.json config: decoder shape + the workload quoted on it."""
    name: str
    d_model: int
    n_layers: int
    n_stages: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    d_ffn: int
    vocab: int
    prompt_len: int
    gen_len: int
    p_sweep: tuple
    rms_eps: float = 1e-6
    rope_base: float = 1e6

    @property
    def max_seq(self) -> int:
        # prompt + generated + in-flight slack (n drafts beyond the last emitted token)
        return self.prompt_len + self.gen_len + 2 * self.n_stages + 8

    def layer_params(self) -> int:
        d, hq, hkv, hd, f = self.d_model, self.n_q_heads, self.n_kv_heads, self.head_dim, self.d_ffn
        return (hq + 2 * hkv) * hd * d + d * hq * hd + 3 * f * d

    def replace(self, **kw) -> "ModelShape":
        return dataclasses.replace(self, **kw)


# BASELINE.json `configs`, in order.  configs[3] ("9b_n4") is the one `metric` is quoted on.
CONFIGS = {
    "tiny": ModelShape("tiny", 256, 8, 2, 4, 2, 64, 704, 1024, 32, 64, ()),
    "4b_n4": ModelShape("4b_n4", 2560, 32, 4, 32, 8, 128, 9728, 151936, 512, 256, (0.6, 0.8, 1.0)),
    "4b_n8": ModelShape("4b_n8", 2560, 32, 8, 32, 8, 128, 9728, 151936, 1024, 256, (0.6, 0.8, 1.0)),
    "9b_n4": ModelShape("9b_n4", 4096, 32, 4, 32, 8, 128, 12288, 151936, 2048, 256, (0.6, 0.8, 1.0)),
    "9b_n16": ModelShape("9b_n16", 4096, 32, 16, 32, 8, 128, 12288, 151936, 4096, 512,
                         (0.4, 0.6, 0.8, 1.0)),
}


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit pattern (uint16), round-to-nearest-even.  Finite inputs only."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    bias = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + bias) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    """bf16 bit pattern (uint16) -> float32, exact."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


_TENSOR_IDS = {"embed": 1, "final_norm": 2, "pdm_proj": 3, "pdm_norm": 4,
               "attn_norm": 10, "wq": 11, "wk": 12, "wv": 13, "wo": 14,
               "mlp_norm": 15, "w_gate": 16, "w_up": 17, "w_down": 18}

def layer_tensor_names():
    return ["attn_norm", "wq", "wk", "wv", "wo", "mlp_norm", "w_gate", "w_up", "w_down"]


def _normal_bf16(seed: int, tid: int, layer: int, n_elem: int, std: float) -> np.ndarray:
    out = np.empty(n_elem, dtype=np.uint16)
    key = (seed * 0x9E3779B97F4A7C15 + tid * 0xD1B54A32D192ED03 + (layer + 1) * 0x2545F4914F6CDD1D) & (2 ** 64 - 1)
    _fastgen().fastgen_normal_bf16(out.ctypes.data, n_elem, key, std)
    return out


def _gain_bf16(seed: int, tid: int, layer: int, d: int, random_gains: bool) -> np.ndarray:
    if not random_gains:
        return np.full(d, 0x3F80, dtype=np.uint16)  # bf16(1.0)
    rng = np.random.Generator(np.random.PCG64([seed, tid, layer + 1, 0]))
    return f32_to_bf16_bits(rng.uniform(0.5, 1.5, d).astype(np.float32))


def shapes_of(shape: ModelShape) -> dict:
    d, hq, hkv, hd, f, v, n = (shape.d_model, shape.n_q_heads, shape.n_kv_heads, shape.head_dim,
                               shape.d_ffn, shape.vocab, shape.n_stages)
    return {"embed": (v, d), "final_norm": (d,), "pdm_proj": (d, n * d), "pdm_norm": (d,),
            "attn_norm": (d,), "wq": (hq * hd, d), "wk": (hkv * hd, d), "wv": (hkv * hd, d),
            "wo": (d, hq * hd), "mlp_norm": (d,), "w_gate": (f, d), "w_up": (f, d),
            "w_down": (d, f)}


def make_tensor(shape: ModelShape, name: str, layer: int, seed: int, std: float = 0.02,
                random_gains: bool = False, scale: float = 1.0) -> np.ndarray:
    """One tensor as a uint16 (bf16 bits) array of its natural [out, in] shape."""
    shp = shapes_of(shape)[name]
    tid = _TENSOR_IDS[name]
    if name.endswith("norm"):
        return _gain_bf16(seed, tid, layer, shp[0], random_gains)
    n_elem = int(np.prod(shp))
    return _normal_bf16(seed, tid, layer, n_elem, std * scale).reshape(shp)


def make_weights(shape: ModelShape, seed: int = 1234, std: float = 0.02, random_gains: bool = False,
                 attention_heavy: bool = False) -> dict:
    """All weights as uint16 (bf16 bits) numpy arrays, row-major [out, in].

    Returns {"embed", "final_norm", "pdm_proj", "pdm_norm", and per-layer lists "attn_norm", "wq",
    "wk", "wv", "wo", "mlp_norm", "w_gate", "w_up", "w_down"}.
    `attention_heavy` (test-only init): W_o and W_v scaled x8, W_d / 8, so that
    attention errors are visible in the hidden state.
    """
    scale = {"wo": 8.0, "wv": 8.0, "w_down": 0.125} if attention_heavy else {}
    w = {}
    for name in ("embed", "final_norm", "pdm_proj", "pdm_norm"):
        w[name] = make_tensor(shape, name, -1, seed, std, random_gains, 1.0)
    for name in layer_tensor_names():
        w[name] = [make_tensor(shape, name, l, seed, std, random_gains, scale.get(name, 1.0))
                   for l in range(shape.n_layers)]
    return w


def pdm_anchor_count(n_layers: int) -> int:
    """How many FC matrices the paper's PDM needs: the anchor list [0, L/4, L/2, 3L/4, L-1] without duplicates (sizes
    only; which layers they are is the method's business and lives on both sides separately)."""
    return len(sorted({0, n_layers // 4, n_layers // 2, (3 * n_layers) // 4, n_layers - 1}))


def make_pdm_weights(shape: ModelShape, pdm_layers: int, pdm_vocab: int, seed: int = 1234, std: float = 0.02,
                     random_gains: bool = False) -> dict:
    """Weights of the paper's Pipeline Draft Module (NEXT-1) as uint16 bf16-bit arrays: "fc" = [m] matrices
    [d, (i+1) d] (std / sqrt(i+1), so every aggregated feature has the scale of one projected state), the nine
    per-layer tensors of `pdm_layers` decoder layers (the target's shapes, own values), "final_norm" [d], "head"
    [pdm_vocab, d], and "vocab_map": int32 [pdm_vocab], a seeded strictly ascending subset of the token ids."""
    d = shape.d_model
    m = pdm_anchor_count(shape.n_layers)
    sp = seed + 7777                                    # the PDM's tensors never alias the target's
    w = {"n_layers": int(pdm_layers), "vocab": int(pdm_vocab)}
    w["fc"] = [_normal_bf16(sp, 20, i, d * (i + 1) * d, std / float(np.sqrt(i + 1))).reshape(d, (i + 1) * d) for i in range(m)]
    for name in layer_tensor_names():
        w[name] = [make_tensor(shape, name, l, sp, std, random_gains, 1.0) for l in range(pdm_layers)]
    w["final_norm"] = _gain_bf16(sp, 22, -1, d, random_gains)
    w["head"] = _normal_bf16(sp, 21, -1, pdm_vocab * d, std).reshape(pdm_vocab, d)
    rng = np.random.Generator(np.random.PCG64([seed, 4711]))
    w["vocab_map"] = np.sort(rng.choice(shape.vocab, size=pdm_vocab, replace=False)).astype(np.int32)
    return w


def make_echo(shape: ModelShape, weights: dict) -> dict:
    """The "echo" re-initialisation used to reach saturation under sampling verification: a copy of
    `weights` with W_o = W_down = 0 (every layer leaves the residual stream untouched), W_p = [I 0 .. 0] (the PDM
    reads the newest token's embedding) and the PDM's norm gain = the final norm's.  The PDM's logits for a token
    then equal the target's logits for it, so the draft distribution equals the target distribution."""
    d, n = shape.d_model, shape.n_stages
    w = dict(weights)
    w["wo"] = [np.zeros_like(x) for x in weights["wo"]]
    w["w_down"] = [np.zeros_like(x) for x in weights["w_down"]]
    proj = np.zeros((d, n * d), dtype=np.uint16)
    proj[np.arange(d), np.arange(d)] = 0x3F80          # bf16 1.0
    w["pdm_proj"] = proj
    w["pdm_norm"] = weights["final_norm"].copy()
    return w


def make_prompt(shape: ModelShape, seed: int = 1, length: int | None = None) -> np.ndarray:
    """Prompt token ids, uniform on [0, vocab), int32."""
    n = shape.prompt_len if length is None else length
    rng = np.random.Generator(np.random.PCG64([seed, 77]))
    return rng.integers(0, shape.vocab, size=n, dtype=np.int32)


def make_kv_filler(shape: ModelShape, layer: int, length: int, seed: int = 5) -> tuple:
    """Seeded random K and V rows ([length, n_kv_heads*head_dim] bf16 bits, ~N(0,1)) used ONLY to
    give a timing run a KV cache of the right length without a prefill (values do not change time)."""
    rng = np.random.Generator(np.random.PCG64([seed, 99, layer]))
    w = shape.n_kv_heads * shape.head_dim
    k = f32_to_bf16_bits(rng.standard_normal((length, w), dtype=np.float32))
    v = f32_to_bf16_bits(rng.standard_normal((length, w), dtype=np.float32))
    return k, v
