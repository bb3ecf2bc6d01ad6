"""ctypes wrapper over oracle/spd_oracle.c.  Argument marshalling only — no arithmetic here."""
from __future__ import annotations

import ctypes as C
from typing import NamedTuple

import numpy as np

from . import build as _build

_LAYER_NAMES = ["attn_norm", "wq", "wk", "wv", "wo", "mlp_norm", "w_gate", "w_up", "w_down"]


class _Cfg(C.Structure):
    _fields_ = [(k, C.c_int32) for k in ("d_model", "n_layers", "n_stages", "n_q_heads", "n_kv_heads",
                                          "head_dim", "d_ffn", "vocab", "max_seq")] + \
               [("rms_eps", C.c_float), ("rope_base", C.c_float)]


_PP = C.POINTER(C.c_void_p)


class _Weights(C.Structure):
    _fields_ = [("embed", C.c_void_p)] + [(k, _PP) for k in _LAYER_NAMES] + \
               [("final_norm", C.c_void_p), ("pdm_proj", C.c_void_p), ("pdm_norm", C.c_void_p)]


class _PdmWeights(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("vocab", C.c_int32), ("fc", _PP)] + [(k, _PP) for k in _LAYER_NAMES] + \
               [("final_norm", C.c_void_p), ("head", C.c_void_p), ("vocab_map", C.c_void_p)]


class _Res(C.Structure):
    _fields_ = [(k, C.c_int32) for k in ("step_index", "fill", "exited", "accepted", "emitted_token",
                                          "draft_token", "draft_forced", "discarded", "committed_len")]


MAX_TOPK = 64


class _Dist(C.Structure):
    _fields_ = [("k", C.c_int32), ("id", C.c_int32 * MAX_TOPK), ("p", C.c_float * MAX_TOPK)]


class _Hints(C.Structure):
    _fields_ = [("draft_k", C.c_int32), ("draft_ids", C.c_int32 * MAX_TOPK),
                ("verify_k", C.c_int32), ("verify_ids", C.c_int32 * MAX_TOPK),
                ("draft_token", C.c_int32), ("accepted", C.c_int32), ("emitted_token", C.c_int32),
                ("logit_band", C.c_float), ("prob_eps", C.c_float)]


class _SampleRec(C.Structure):
    _fields_ = [("draft", _Dist), ("target", _Dist),
                ("u_draft", C.c_double), ("u_accept", C.c_double), ("u_resid", C.c_double),
                ("succ_token", C.c_int32), ("succ_q", C.c_float), ("succ_p", C.c_float),
                ("ties_support", C.c_int32), ("ties_draft", C.c_int32), ("ties_accept", C.c_int32),
                ("ties_resid", C.c_int32)]


class Dist(NamedTuple):
    """A filtered distribution: support in ascending token id, fp32 probabilities."""
    ids: np.ndarray
    p: np.ndarray


def _dist_out(d: _Dist) -> Dist:
    k = d.k
    return Dist(np.array(d.id[:k], dtype=np.int32), np.array(d.p[:k], dtype=np.float32))


def _dist_in(d: Dist) -> _Dist:
    out = _Dist()
    out.k = len(d.ids)
    for i, (t, p) in enumerate(zip(d.ids, d.p)):
        out.id[i] = int(t)
        out.p[i] = float(p)
    return out


class StepResult(NamedTuple):
    step_index: int
    fill: int
    exited: int
    accepted: int
    emitted_token: int
    draft_token: int
    draft_forced: int
    discarded: int
    committed_len: int


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.ora_create.restype = C.c_void_p
        L.ora_create.argtypes = [C.POINTER(_Cfg), C.POINTER(_Weights)]
        L.ora_destroy.argtypes = [C.c_void_p]
        L.ora_prefill.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.POINTER(C.c_int32)]
        L.ora_step.argtypes = [C.c_void_p, C.c_int32, C.POINTER(_Res)]
        L.ora_step_follow.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_float, C.POINTER(_Res)]
        L.ora_get_ties.argtypes = [C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.ora_rollback.argtypes = [C.c_void_p, C.c_int32, C.c_int32]
        L.ora_set_forced.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_float, C.c_uint64]
        L.ora_ar_step.argtypes = [C.c_void_p, C.POINTER(C.c_int32)]
        L.ora_ar_set_trace.argtypes = [C.c_void_p, C.c_void_p]
        L.ora_set_forward_order.argtypes = [C.c_void_p, C.c_int32]
        L.ora_committed_len.argtypes = [C.c_void_p]
        L.ora_fill.argtypes = [C.c_void_p]
        L.ora_steps.argtypes = [C.c_void_p]
        L.ora_steps.restype = C.c_int64
        L.ora_emitted.argtypes = [C.c_void_p]
        L.ora_get_kv_len.argtypes = [C.c_void_p, C.c_void_p]
        L.ora_get_kv.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p]
        L.ora_get_ring.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_int32), C.POINTER(C.c_int32),
                                   C.POINTER(C.c_int32), C.c_void_p]
        L.ora_get_hfin.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
        L.ora_get_last.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
        L.ora_get_margin.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_float), C.POINTER(C.c_float)]
        L.ora_load_kv.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_int32]
        L.ora_assume_prefilled.argtypes = [C.c_void_p, C.c_int32, C.c_int32]
        L.ora_op_rmsnorm.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_float, C.c_void_p]
        L.ora_op_gemv.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        L.ora_op_rope.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_float]
        L.ora_op_attention.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int32,
                                       C.c_int32, C.c_void_p]
        L.ora_op_silu_mul.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
        L.ora_op_argmax.argtypes = [C.c_void_p, C.c_int32]
        L.ora_op_f32_to_bf16.argtypes = [C.c_float]
        L.ora_op_f32_to_bf16.restype = C.c_uint16
        L.ora_op_splitmix64.argtypes = [C.c_uint64]
        L.ora_op_splitmix64.restype = C.c_uint64
        L.ora_num_threads.restype = C.c_int32
        L.ora_op_topk_softmax.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_float, C.c_void_p, C.POINTER(_Dist)]
        L.ora_op_uniform.argtypes = [C.c_uint64, C.c_int64, C.c_int32]
        L.ora_op_uniform.restype = C.c_double
        L.ora_op_sample_cdf.argtypes = [C.POINTER(_Dist), C.c_double]
        L.ora_op_accept.argtypes = [C.POINTER(_Dist), C.POINTER(_Dist), C.c_int32, C.c_double]
        L.ora_op_sample_residual.argtypes = [C.POINTER(_Dist), C.POINTER(_Dist), C.c_double]
        L.ora_set_sampling.argtypes = [C.c_void_p, C.c_float, C.c_int32, C.c_uint64]
        L.ora_step_sample_follow.argtypes = [C.c_void_p, C.c_int32, C.POINTER(_Hints), C.POINTER(_Res)]
        L.ora_get_sample_record.argtypes = [C.c_void_p, C.POINTER(_SampleRec)]
        L.ora_pdm_attach.argtypes = [C.c_void_p, C.POINTER(_PdmWeights)]
        L.ora_pdm_anchors.argtypes = [C.c_void_p, C.c_void_p]
        L.ora_pdm_f.argtypes = [C.c_void_p, C.c_int32]
        L.ora_pdm_get_anchor.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p]
        L.ora_pdm_get_last.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
        L.ora_pdm_last_rows.argtypes = [C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.c_void_p]
        L.ora_pdm_get_kv.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.POINTER(C.c_int32)]
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _u16(a) -> np.ndarray:
    a = np.ascontiguousarray(a)
    assert a.dtype == np.uint16, a.dtype
    return a


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


class Oracle:
    """One oracle context.  `shape` is a spd_inputs.ModelShape (or anything with the same fields);
    `weights` is the dict spd_inputs.make_weights returns (uint16 bf16-bit arrays)."""

    def __init__(self, shape, weights, max_seq: int | None = None):
        self.shape = shape
        self.max_seq = int(max_seq if max_seq is not None else shape.max_seq)
        self._keep = []
        cfg = _Cfg(shape.d_model, shape.n_layers, shape.n_stages, shape.n_q_heads, shape.n_kv_heads,
                   shape.head_dim, shape.d_ffn, shape.vocab, self.max_seq, shape.rms_eps, shape.rope_base)
        w = _Weights()
        for name in ("embed", "final_norm", "pdm_proj", "pdm_norm"):
            arr = _u16(weights[name])
            self._keep.append(arr)
            setattr(w, name, arr.ctypes.data)
        for name in _LAYER_NAMES:
            arrs = [_u16(x) for x in weights[name]]
            self._keep.extend(arrs)
            tab = (C.c_void_p * len(arrs))(*[x.ctypes.data for x in arrs])
            self._keep.append(tab)
            setattr(w, name, C.cast(tab, _PP))
        self._h = lib().ora_create(C.byref(cfg), C.byref(w))
        if not self._h:
            raise ValueError("ora_create rejected the configuration")

    def close(self):
        if self._h:
            lib().ora_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- path ------------------------------------------------------------------------------
    def prefill(self, tokens, block: int = 1) -> int:
        t = np.ascontiguousarray(tokens, dtype=np.int32)
        first = C.c_int32(-1)
        rc = lib().ora_prefill(self._h, _p(t), len(t), block, C.byref(first))
        if rc:
            raise RuntimeError(f"ora_prefill rc={rc}")
        return first.value

    def step(self, draft_override: int = -1) -> StepResult:
        r = _Res()
        rc = lib().ora_step(self._h, draft_override, C.byref(r))
        if rc:
            raise RuntimeError(f"ora_step rc={rc}")
        return StepResult(*[getattr(r, k) for k, _ in _Res._fields_])

    def step_follow(self, draft_hint: int, verify_hint: int, band: float) -> StepResult:
        r = _Res()
        rc = lib().ora_step_follow(self._h, -1, draft_hint, verify_hint, band, C.byref(r))
        if rc:
            raise RuntimeError(f"ora_step_follow rc={rc}")
        return StepResult(*[getattr(r, k) for k, _ in _Res._fields_])

    def ties(self):
        v, p = C.c_int32(), C.c_int32()
        lib().ora_get_ties(self._h, C.byref(v), C.byref(p))
        return v.value, p.value

    def rollback(self, new_len: int, reseed_token: int) -> int:
        return lib().ora_rollback(self._h, new_len, reseed_token)

    def set_forced(self, truth, p: float, seed: int):
        if truth is None:
            rc = lib().ora_set_forced(self._h, None, 0, p, seed)
        else:
            t = np.ascontiguousarray(truth, dtype=np.int32)
            self._keep.append(t)
            rc = lib().ora_set_forced(self._h, _p(t), len(t), p, seed)
        if rc:
            raise ValueError("ora_set_forced")

    def set_sampling(self, temperature: float, top_k: int, seed: int):
        if lib().ora_set_sampling(self._h, temperature, top_k, seed):
            raise ValueError("ora_set_sampling")

    def step_sample_follow(self, draft_ids=None, verify_ids=None, draft_token: int = -1, accepted: int = -1,
                           emitted_token: int = -1, logit_band: float = 0.0, prob_eps: float = 0.0,
                           draft_override: int = -1) -> StepResult:
        h = _Hints()
        for name, ids in (("draft", draft_ids), ("verify", verify_ids)):
            n = 0 if ids is None else len(ids)
            setattr(h, name + "_k", n)
            for i in range(n):
                getattr(h, name + "_ids")[i] = int(ids[i])
        h.draft_token, h.accepted, h.emitted_token = draft_token, accepted, emitted_token
        h.logit_band, h.prob_eps = logit_band, prob_eps
        r = _Res()
        rc = lib().ora_step_sample_follow(self._h, draft_override, C.byref(h), C.byref(r))
        if rc:
            raise RuntimeError(f"ora_step_sample_follow rc={rc}")
        return StepResult(*[getattr(r, k) for k, _ in _Res._fields_])

    def sample_record(self) -> dict:
        r = _SampleRec()
        lib().ora_get_sample_record(self._h, C.byref(r))
        return dict(draft=_dist_out(r.draft), target=_dist_out(r.target), u_draft=r.u_draft, u_accept=r.u_accept,
                    u_resid=r.u_resid, succ_token=r.succ_token, succ_q=r.succ_q, succ_p=r.succ_p,
                    ties=(r.ties_support, r.ties_draft, r.ties_accept, r.ties_resid))

    # -- NEXT-1: the paper's PDM -------------------------------------------------------------
    def attach_pdm(self, pw: dict):
        """pw = spd_inputs.make_pdm_weights(...).  Before prefill."""
        w = _PdmWeights()
        w.n_layers, w.vocab = pw["n_layers"], pw["vocab"]
        self.pdm_vocab = pw["vocab"]
        for name in ["fc"] + _LAYER_NAMES:
            arrs = [_u16(x) for x in pw[name]]
            self._keep.extend(arrs)
            tab = (C.c_void_p * len(arrs))(*[x.ctypes.data for x in arrs])
            self._keep.append(tab)
            setattr(w, name, C.cast(tab, _PP))
        for name in ("final_norm", "head"):
            arr = _u16(pw[name])
            self._keep.append(arr)
            setattr(w, name, arr.ctypes.data)
        vm = np.ascontiguousarray(pw["vocab_map"], dtype=np.int32)
        self._keep.append(vm)
        w.vocab_map = vm.ctypes.data
        if lib().ora_pdm_attach(self._h, C.byref(w)):
            raise ValueError("ora_pdm_attach")

    def pdm_anchors(self) -> list:
        b = np.zeros(8, dtype=np.int32)
        m = lib().ora_pdm_anchors(self._h, _p(b))
        return [int(x) for x in b[:m]]

    def pdm_f(self, k: int) -> int:
        return lib().ora_pdm_f(self._h, k)

    def pdm_anchor(self, pos: int, i: int) -> np.ndarray:
        out = np.zeros(self.shape.d_model, dtype=np.float32)
        lib().ora_pdm_get_anchor(self._h, pos, i, _p(out))
        return out

    def pdm_rows(self):
        """(first position, per-row depths k) of the last PDM run."""
        first, rows = C.c_int32(), C.c_int32()
        lib().ora_pdm_last_rows(self._h, C.byref(first), C.byref(rows), None)
        depths = np.zeros(rows.value, dtype=np.int32)
        lib().ora_pdm_last_rows(self._h, C.byref(first), C.byref(rows), _p(depths))
        return first.value, depths

    def pdm_last(self, what: str) -> np.ndarray:
        first, depths = self.pdm_rows()
        idx = {"logits": 0, "hidden": 1, "features": 2}[what]
        n = {0: self.pdm_vocab, 1: self.shape.d_model, 2: len(depths) * self.shape.d_model}[idx]
        out = np.zeros(n, dtype=np.float32)
        lib().ora_pdm_get_last(self._h, idx, _p(out))
        return out.reshape(len(depths), -1) if idx == 2 else out

    def pdm_kv(self, layer: int, which: int, rows: int):
        out = np.zeros((rows, self.shape.n_kv_heads * self.shape.head_dim), dtype=np.uint16)
        fin = C.c_int32()
        lib().ora_pdm_get_kv(self._h, layer, which, rows, _p(out), C.byref(fin))
        return out, fin.value

    def ar_step(self) -> int:
        nxt = C.c_int32(-1)
        rc = lib().ora_ar_step(self._h, C.byref(nxt))
        if rc:
            raise RuntimeError(f"ora_ar_step rc={rc}")
        return nxt.value

    def ar_set_trace(self, enable: bool = True):
        if enable:
            self._trace = np.zeros((self.shape.n_layers + 1, self.shape.d_model), dtype=np.float32)
            lib().ora_ar_set_trace(self._h, _p(self._trace))
        else:
            self._trace = None
            lib().ora_ar_set_trace(self._h, None)
        return self._trace

    def set_forward_order(self, reverse: bool):
        lib().ora_set_forward_order(self._h, int(reverse))

    def generate_spd(self, n_tokens: int, draft_fn=None, max_steps: int | None = None):
        """Run cycles until n_tokens tokens are emitted (the prefill's first token counts).
        Returns (emitted tokens excluding the first, list of StepResult)."""
        out, log = [], []
        limit = max_steps if max_steps is not None else 10 ** 9
        while lib().ora_emitted(self._h) < n_tokens and len(log) < limit:
            ov = -1 if draft_fn is None else int(draft_fn(self))
            r = self.step(ov)
            log.append(r)
            if r.exited:
                out.append(r.emitted_token)
        return out, log

    # -- readers ---------------------------------------------------------------------------
    @property
    def committed_len(self) -> int:
        return lib().ora_committed_len(self._h)

    @property
    def fill(self) -> int:
        return lib().ora_fill(self._h)

    @property
    def steps(self) -> int:
        return lib().ora_steps(self._h)

    @property
    def emitted(self) -> int:
        return lib().ora_emitted(self._h)

    def kv_len(self) -> np.ndarray:
        out = np.zeros(self.shape.n_layers, dtype=np.int32)
        lib().ora_get_kv_len(self._h, _p(out))
        return out

    def kv(self, layer: int, which: int, rows: int) -> np.ndarray:
        out = np.zeros((rows, self.shape.n_kv_heads * self.shape.head_dim), dtype=np.uint16)
        if rows:
            lib().ora_get_kv(self._h, layer, which, rows, _p(out))
        return out

    def ring(self, i: int):
        pos, tok, k = C.c_int32(), C.c_int32(), C.c_int32()
        h = np.zeros(self.shape.d_model, dtype=np.float32)
        rc = lib().ora_get_ring(self._h, i, C.byref(pos), C.byref(tok), C.byref(k), _p(h))
        if rc:
            raise IndexError(i)
        return pos.value, tok.value, k.value, h

    def hfin(self, pos: int) -> np.ndarray:
        out = np.zeros(self.shape.d_model, dtype=np.float32)
        lib().ora_get_hfin(self._h, pos, _p(out))
        return out

    def last(self, what: str) -> np.ndarray:
        idx = {"exit_logits": 0, "pdm_logits": 1, "pdm_prenorm": 2, "pdm_feat": 3}[what]
        n = {0: self.shape.vocab, 1: self.shape.vocab, 2: self.shape.d_model,
             3: self.shape.d_model * self.shape.n_stages}[idx]
        out = np.zeros(n, dtype=np.float32)
        lib().ora_get_last(self._h, idx, _p(out))
        return out

    def margin(self, which: int):
        g, m = C.c_float(), C.c_float()
        lib().ora_get_margin(self._h, which, C.byref(g), C.byref(m))
        return g.value, m.value

    # -- timing-only -----------------------------------------------------------------------
    def load_kv(self, layer: int, k: np.ndarray, v: np.ndarray):
        k, v = _u16(k), _u16(v)
        lib().ora_load_kv(self._h, layer, _p(k), _p(v), k.shape[0])

    def assume_prefilled(self, committed_len: int, first_token: int):
        if lib().ora_assume_prefilled(self._h, committed_len, first_token):
            raise ValueError("ora_assume_prefilled")


# -- single operations (per-kernel parity) -----------------------------------------------------

def op_rmsnorm(x, gain, eps: float) -> np.ndarray:
    x, gain = _f32(x), _u16(gain)
    out = np.empty_like(x)
    lib().ora_op_rmsnorm(_p(x), _p(gain), x.size, eps, _p(out))
    return out


def op_gemv(w, x) -> np.ndarray:
    w, x = _u16(w), _f32(x)
    rows, k = w.shape
    assert x.size == k
    out = np.empty(rows, dtype=np.float32)
    lib().ora_op_gemv(_p(w), rows, k, _p(x), _p(out))
    return out


def op_rope(vec, n_heads: int, head_dim: int, pos: int, base: float) -> np.ndarray:
    v = _f32(vec).copy()
    lib().ora_op_rope(_p(v), n_heads, head_dim, pos, base)
    return v


def op_attention(q, kc, vc, n_q_heads: int, n_kv_heads: int, head_dim: int) -> np.ndarray:
    q, kc, vc = _f32(q), _u16(kc), _u16(vc)
    out = np.empty(n_q_heads * head_dim, dtype=np.float32)
    lib().ora_op_attention(_p(q), _p(kc), _p(vc), kc.shape[0], n_q_heads, n_kv_heads, head_dim, _p(out))
    return out


def op_silu_mul(gate, up) -> np.ndarray:
    g, u = _f32(gate), _f32(up)
    out = np.empty_like(g)
    lib().ora_op_silu_mul(_p(g), _p(u), g.size, _p(out))
    return out


def op_argmax(x) -> int:
    x = _f32(x)
    return lib().ora_op_argmax(_p(x), x.size)


def op_f32_to_bf16(x: float) -> int:
    return lib().ora_op_f32_to_bf16(x)


def op_splitmix64(x: int) -> int:
    return lib().ora_op_splitmix64(x & 0xFFFFFFFFFFFFFFFF)


def num_threads() -> int:
    return lib().ora_num_threads()


# -- NEXT-2 sampling operations ------------------------------------------------------------------

def op_topk_softmax(logits, top_k: int, temperature: float, support=None) -> Dist:
    x = _f32(logits)
    d = _Dist()
    sup = None if support is None else np.ascontiguousarray(support, dtype=np.int32)
    lib().ora_op_topk_softmax(_p(x), x.size, top_k, temperature, None if sup is None else _p(sup), C.byref(d))
    return _dist_out(d)


def op_uniform(seed: int, K: int, j: int) -> float:
    return lib().ora_op_uniform(seed & 0xFFFFFFFFFFFFFFFF, K, j)


def op_sample_cdf(dist: Dist, u: float) -> int:
    return lib().ora_op_sample_cdf(C.byref(_dist_in(dist)), u)


def op_accept(P: Dist, Q: Dist, token: int, u: float) -> int:
    return lib().ora_op_accept(C.byref(_dist_in(P)), C.byref(_dist_in(Q)), token, u)


def op_sample_residual(P: Dist, Q: Dist, u: float) -> int:
    return lib().ora_op_sample_residual(C.byref(_dist_in(P)), C.byref(_dist_in(Q)), u)
