"""ctypes binding of include/spd.h.  Same names as the C ABI; argument marshalling only.

PyTorch is used for device memory and streams (torch.empty / torch.cuda.Stream); the library never
allocates device memory itself.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import NamedTuple

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libspd_b200.so")
_LAYER_NAMES = ["attn_norm", "wq", "wk", "wv", "wo", "mlp_norm", "w_gate", "w_up", "w_down"]


class SpdError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"spd status {status} ({_STATUS.get(status, '?')}): {msg}")
        self.status = status


_STATUS = {0: "SPD_OK", 1: "SPD_EINVAL", 2: "SPD_ESTATE", 3: "SPD_ECAPACITY", 4: "SPD_ECUDA", 5: "SPD_ENOMEM"}


class OPT:
    ENGINE = 0
    DEBUG_LOGITS = 1
    PHASE_PROFILE = 2
    PREFILL = 3
    CHAINS = 4


class DBG:
    SLOT_HIDDEN, EXIT_LOGITS, PDM_LOGITS, PDM_PRENORM, PDM_FEAT, KV_K, KV_V, KV_LEN, RING, HFIN, PHASE_PROFILE, \
        SAMPLE, Q, ATT, CYCLE_TIMES, PDM2_LOGITS, PDM2_HIDDEN, PDM2_RUN, PDM2_FEAT, PDM2_K, PDM2_V, ANCHOR = range(22)


MAX_TOPK = 64


class _Dist(C.Structure):
    _fields_ = [("k", C.c_int32), ("id", C.c_int32 * MAX_TOPK), ("p", C.c_float * MAX_TOPK)]


class _SampleRec(C.Structure):
    _fields_ = [("draft", _Dist), ("target", _Dist), ("u_draft", C.c_float), ("u_accept", C.c_float),
                ("u_resid", C.c_float), ("succ_token", C.c_int32), ("succ_q", C.c_float), ("succ_p", C.c_float),
                ("exact_rounds", C.c_int32), ("prefiltered", C.c_int32)]


def _dist_out(d: _Dist):
    k = d.k
    return np.array(d.id[:k], dtype=np.int32), np.array(d.p[:k], dtype=np.float32)


class _Cfg(C.Structure):
    _fields_ = [(k, C.c_int32) for k in ("d_model", "n_layers", "n_stages", "n_q_heads", "n_kv_heads",
                                          "head_dim", "d_ffn", "vocab", "max_seq")] + \
               [("rms_eps", C.c_float), ("rope_base", C.c_float), ("device", C.c_int32)]


_PP = C.POINTER(C.c_void_p)


class _Weights(C.Structure):
    _fields_ = [("embed", C.c_void_p)] + [(k, _PP) for k in _LAYER_NAMES] + \
               [("final_norm", C.c_void_p), ("pdm_proj", C.c_void_p), ("pdm_norm", C.c_void_p)]


class _Sizes(C.Structure):
    _fields_ = [("repack_bytes", C.c_size_t), ("kv_bytes", C.c_size_t), ("work_bytes", C.c_size_t)]


class _Buffers(C.Structure):
    _fields_ = [("repack", C.c_void_p), ("kv", C.c_void_p), ("work", C.c_void_p),
                ("stream_main", C.c_void_p), ("stream_pdm", C.c_void_p),
                ("repack_bytes", C.c_size_t), ("kv_bytes", C.c_size_t), ("work_bytes", C.c_size_t)]


class _PdmWeights(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("vocab", C.c_int32), ("fc", _PP)] + [(k, _PP) for k in _LAYER_NAMES] + \
               [("final_norm", C.c_void_p), ("head", C.c_void_p), ("vocab_map", C.c_void_p)]


class _PdmSizes(C.Structure):
    _fields_ = [("kv_bytes", C.c_size_t), ("work_bytes", C.c_size_t)]


class _Res(C.Structure):
    _fields_ = [(k, C.c_int32) for k in ("step_index", "fill", "exited", "accepted", "emitted_token",
                                          "draft_token", "draft_forced", "discarded", "committed_len")]


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


_RES_KEYS = [k for k, _ in _Res._fields_]
_lib = None


def lib():
    """Loads libspd_b200.so.  Fails loudly if it is missing — there is no fallback path."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError(f"{_LIB_PATH} is missing: build the CUDA library first "
                              "(python -m paper_2605_30852_b200.build, or __graft_entry__.build())")
        L = C.CDLL(_LIB_PATH)
        vp, i32, f32, u64 = C.c_void_p, C.c_int32, C.c_float, C.c_uint64
        L.spd_query_sizes.argtypes = [C.POINTER(_Cfg), C.POINTER(_Sizes)]
        L.spd_create.argtypes = [C.POINTER(_Cfg), C.POINTER(_Weights), C.POINTER(_Buffers), C.POINTER(vp)]
        L.spd_destroy.argtypes = [vp]
        L.spd_prefill.argtypes = [vp, vp, i32, C.POINTER(i32)]
        L.spd_step.argtypes = [vp, C.POINTER(_Res)]
        L.spd_step_many.argtypes = [vp, i32, C.POINTER(_Res)]
        L.spd_rollback.argtypes = [vp, i32, i32]
        L.spd_set_forced.argtypes = [vp, vp, i32, f32, u64]
        L.spd_set_option.argtypes = [vp, i32, i32]
        L.spd_get_option.argtypes = [vp, i32, C.POINTER(i32)]
        L.spd_set_sampling.argtypes = [vp, f32, i32, u64]
        L.spd_op_topk_softmax.argtypes = [vp, i32, i32, f32, i32, vp, vp, vp]
        L.spd_op_topk_scratch.argtypes = []
        L.spd_op_topk_scratch.restype = C.c_size_t
        L.spd_debug_read.argtypes = [vp, i32, i32, vp, C.c_size_t]
        L.spd_get_counters.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.spd_last_error.argtypes = [vp]
        L.spd_last_error.restype = C.c_char_p
        L.spd_op_rmsnorm.argtypes = [vp, vp, i32, f32, vp, vp]
        L.spd_op_gemv.argtypes = [vp, i32, i32, vp, vp, vp]
        L.spd_op_gemm.argtypes = [vp, vp, i32, i32, i32, vp, vp, vp]
        L.spd_op_gemm_scratch.argtypes = [i32, i32]
        L.spd_op_gemm_scratch.restype = C.c_size_t
        L.spd_pdm_query_sizes.argtypes = [vp, i32, i32, vp]
        L.spd_pdm_attach.argtypes = [vp, vp, vp, vp]
        L.spd_op_rope.argtypes = [vp, i32, i32, i32, f32, vp]
        L.spd_op_attention.argtypes = [vp, vp, vp, i32, i32, i32, i32, i32, vp, vp, vp]
        L.spd_op_attention_scratch.argtypes = [i32, i32, i32]
        L.spd_op_attention_scratch.restype = C.c_size_t
        L.spd_op_attention_static.argtypes = [vp, vp, vp, i32, i32, i32, i32, i32, vp, vp]
        L.spd_op_attention_static_max_bytes.argtypes = []
        L.spd_op_attention_static_max_bytes.restype = C.c_size_t
        L.spd_op_silu_mul.argtypes = [vp, vp, i32, vp, vp]
        L.spd_op_argmax.argtypes = [vp, i32, vp, vp]
        _lib = L
    return _lib


def upload_weights(weights: dict, device: int = 0) -> dict:
    """uint16 (bf16 bits) numpy arrays -> int16 CUDA tensors of the same bytes and shapes."""
    dev = torch.device("cuda", device)

    def up(a):
        return torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).to(dev)

    out = {}
    for k, v in weights.items():
        out[k] = [up(x) for x in v] if isinstance(v, (list, tuple)) else up(v)
    return out


def upload_pdm_weights(pw: dict, device: int = 0) -> dict:
    """spd_inputs.make_pdm_weights(...) -> CUDA tensors (bf16 bits as int16; vocab_map int32)."""
    dev = torch.device("cuda", device)

    def up(a):
        return torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).to(dev)

    out = {"n_layers": int(pw["n_layers"]), "vocab": int(pw["vocab"]),
           "vocab_map": torch.from_numpy(np.ascontiguousarray(pw["vocab_map"], dtype=np.int32)).to(dev)}
    for k, v in pw.items():
        if k in out:
            continue
        out[k] = [up(x) for x in v] if isinstance(v, (list, tuple)) else up(v)
    return out


def _cfg_of(shape, max_seq: int, device: int) -> _Cfg:
    return _Cfg(shape.d_model, shape.n_layers, shape.n_stages, shape.n_q_heads, shape.n_kv_heads,
                shape.head_dim, shape.d_ffn, shape.vocab, max_seq, shape.rms_eps, shape.rope_base, device)


def query_sizes(shape, max_seq: int | None = None, device: int = 0):
    cfg = _cfg_of(shape, int(max_seq if max_seq is not None else shape.max_seq), device)
    s = _Sizes()
    rc = lib().spd_query_sizes(C.byref(cfg), C.byref(s))
    if rc:
        raise SpdError(rc, "spd_query_sizes")
    return s.repack_bytes, s.kv_bytes, s.work_bytes


class SPD:
    """One spd_ctx.  `dev_weights`: dict of CUDA tensors (2-byte dtype) as upload_weights returns."""

    def __init__(self, shape, dev_weights: dict, max_seq: int | None = None, device: int = 0):
        L = lib()
        self.shape = shape
        self.device = device
        self.max_seq = int(max_seq if max_seq is not None else shape.max_seq)
        self._w = dev_weights
        cfg = _cfg_of(shape, self.max_seq, device)
        sizes = _Sizes()
        rc = L.spd_query_sizes(C.byref(cfg), C.byref(sizes))
        if rc:
            raise SpdError(rc, "spd_query_sizes: unsupported configuration")
        if not torch.cuda.is_available():
            raise SpdError(4, "no CUDA device: the SPD path has no CPU fallback")
        dev = torch.device("cuda", device)
        self._repack = torch.empty(max(sizes.repack_bytes, 256), dtype=torch.uint8, device=dev)
        self._kv = torch.zeros(sizes.kv_bytes, dtype=torch.uint8, device=dev)
        self._work = torch.empty(sizes.work_bytes, dtype=torch.uint8, device=dev)
        self.stream_main = torch.cuda.Stream(device=dev)
        self.stream_pdm = torch.cuda.Stream(device=dev)
        self.sizes = (sizes.repack_bytes, sizes.kv_bytes, sizes.work_bytes)
        w = _Weights()
        self._tabs = []
        for name in ("embed", "final_norm", "pdm_proj", "pdm_norm"):
            t = dev_weights[name]
            assert t.is_cuda and t.element_size() == 2 and t.is_contiguous()
            setattr(w, name, t.data_ptr())
        for name in _LAYER_NAMES:
            ts = dev_weights[name]
            assert len(ts) == shape.n_layers and all(t.is_cuda and t.is_contiguous() for t in ts)
            tab = (C.c_void_p * len(ts))(*[t.data_ptr() for t in ts])
            self._tabs.append(tab)
            setattr(w, name, C.cast(tab, _PP))
        bufs = _Buffers(self._repack.data_ptr(), self._kv.data_ptr(), self._work.data_ptr(),
                        self.stream_main.cuda_stream, self.stream_pdm.cuda_stream,
                        self._repack.numel(), self._kv.numel(), self._work.numel())
        torch.cuda.synchronize(dev)
        h = C.c_void_p()
        rc = L.spd_create(C.byref(cfg), C.byref(w), C.byref(bufs), C.byref(h))
        if rc:
            raise SpdError(rc, "spd_create")
        self._h = h

    # ------------------------------------------------------------------ plumbing
    def _check(self, rc: int):
        if rc:
            raise SpdError(rc, lib().spd_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            lib().spd_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ------------------------------------------------------------------ NEXT-1: the paper's PDM
    def attach_pdm(self, dev_pdm: dict):
        """dev_pdm = upload_pdm_weights(spd_inputs.make_pdm_weights(...)).  Before prefill."""
        cfg = _cfg_of(self.shape, self.max_seq, self.device)
        sz = _PdmSizes()
        self._check(lib().spd_pdm_query_sizes(C.byref(cfg), dev_pdm["n_layers"], dev_pdm["vocab"], C.byref(sz)))
        dev = torch.device("cuda", self.device)
        self._pdm_kv = torch.zeros(sz.kv_bytes, dtype=torch.uint8, device=dev)
        self._pdm_work = torch.empty(sz.work_bytes, dtype=torch.uint8, device=dev)
        self._pdm_w = dev_pdm
        self.pdm_vocab = dev_pdm["vocab"]
        w = _PdmWeights()
        w.n_layers, w.vocab = dev_pdm["n_layers"], dev_pdm["vocab"]
        for name in ["fc"] + _LAYER_NAMES:
            ts = dev_pdm[name]
            assert all(t.is_cuda and t.is_contiguous() and t.element_size() == 2 for t in ts)
            tab = (C.c_void_p * len(ts))(*[t.data_ptr() for t in ts])
            self._tabs.append(tab)
            setattr(w, name, C.cast(tab, _PP))
        w.final_norm, w.head = dev_pdm["final_norm"].data_ptr(), dev_pdm["head"].data_ptr()
        assert dev_pdm["vocab_map"].dtype == torch.int32
        w.vocab_map = dev_pdm["vocab_map"].data_ptr()
        torch.cuda.synchronize(dev)
        self._check(lib().spd_pdm_attach(self._h, C.byref(w), self._pdm_kv.data_ptr(), self._pdm_work.data_ptr()))

    def pdm_run(self):
        """(first position, rows, F) of the paper PDM's last draft."""
        r = self.debug_read(DBG.PDM2_RUN, 0, np.int32, 3)
        return int(r[0]), int(r[1]), int(r[2])

    def pdm_last(self, what: str) -> np.ndarray:
        if what == "logits":
            return self.debug_read(DBG.PDM2_LOGITS, 0, np.float32, self.pdm_vocab)
        if what == "hidden":
            return self.debug_read(DBG.PDM2_HIDDEN, 0, np.float32, self.shape.d_model)
        rows = self.pdm_run()[1]
        return self.debug_read(DBG.PDM2_FEAT, rows, np.float32, rows * self.shape.d_model).reshape(rows, -1)

    def pdm_kv(self, layer: int, which: int, rows: int) -> np.ndarray:
        w = self.shape.n_kv_heads * self.shape.head_dim
        return self.debug_read(DBG.PDM2_V if which else DBG.PDM2_K, layer, np.uint16, rows * w).reshape(rows, w)

    def anchor(self, pos: int, i: int) -> np.ndarray:
        return self.debug_read(DBG.ANCHOR, pos * 8 + i, np.float32, self.shape.d_model)

    # ------------------------------------------------------------------ the path
    def prefill(self, tokens) -> int:
        t = np.ascontiguousarray(tokens, dtype=np.int32)
        first = C.c_int32(-1)
        self._check(lib().spd_prefill(self._h, t.ctypes.data, len(t), C.byref(first)))
        return first.value

    def step(self) -> StepResult:
        r = _Res()
        self._check(lib().spd_step(self._h, C.byref(r)))
        return StepResult(*[getattr(r, k) for k in _RES_KEYS])

    def step_many(self, n: int):
        arr = (_Res * n)()
        self._check(lib().spd_step_many(self._h, n, arr))
        return [StepResult(*[getattr(r, k) for k in _RES_KEYS]) for r in arr]

    def rollback(self, new_len: int, reseed_token: int):
        self._check(lib().spd_rollback(self._h, new_len, reseed_token))

    def set_forced(self, truth, p: float, seed: int):
        if truth is None or p < 0:
            self._check(lib().spd_set_forced(self._h, None, 0, -1.0, 0))
        else:
            t = np.ascontiguousarray(truth, dtype=np.int32)
            self._check(lib().spd_set_forced(self._h, t.ctypes.data, len(t), p, seed))

    def set_sampling(self, temperature: float, top_k: int, seed: int):
        """Sampling verification (include/spd.h spd_set_sampling); top_k < 1 switches back to greedy."""
        self._check(lib().spd_set_sampling(self._h, temperature, top_k, seed))

    def sample_record(self) -> dict:
        """spd_sample_record of the last cycle: (ids, p) of the draft and target distributions, the uniforms,
        the judged token with its two probabilities."""
        r = _SampleRec()
        self._check(lib().spd_debug_read(self._h, DBG.SAMPLE, 0, C.addressof(r), C.sizeof(r)))
        return dict(draft=_dist_out(r.draft), target=_dist_out(r.target), u_draft=r.u_draft, u_accept=r.u_accept,
                    u_resid=r.u_resid, succ_token=r.succ_token, succ_q=r.succ_q, succ_p=r.succ_p,
                    exact_rounds=r.exact_rounds, prefiltered=r.prefiltered)

    def set_option(self, option: int, value: int):
        self._check(lib().spd_set_option(self._h, option, value))

    def get_option(self, option: int) -> int:
        v = C.c_int32()
        self._check(lib().spd_get_option(self._h, option, C.byref(v)))
        return int(v.value)

    def counters(self):
        k, n, l = C.c_int64(), C.c_int64(), C.c_int64()
        self._check(lib().spd_get_counters(self._h, C.byref(k), C.byref(n), C.byref(l)))
        return k.value, n.value, l.value

    def generate(self, n_tokens: int, chunk: int = 1):
        """Cycles until n_tokens tokens are emitted (the prefill's first token counts).
        Returns (emitted tokens excluding the first, list of StepResult)."""
        out, log = [], []
        emitted = self.counters()[1]
        while emitted < n_tokens:
            rs = self.step_many(chunk) if chunk > 1 else [self.step()]
            for r in rs:
                log.append(r)
                if r.exited:
                    out.append(r.emitted_token)
                    emitted += 1
        return out, log

    # ------------------------------------------------------------------ debug readers
    def debug_read(self, what: int, index: int, dtype, count: int) -> np.ndarray:
        out = np.zeros(count, dtype=dtype)
        self._check(lib().spd_debug_read(self._h, what, index, out.ctypes.data, out.nbytes))
        return out

    def ring(self):
        """(fill, committed_len, [(occupied, pos, tok) per depth k])."""
        n = self.shape.n_stages
        r = self.debug_read(DBG.RING, 0, np.int32, 2 + 3 * n)
        return int(r[0]), int(r[1]), [tuple(int(v) for v in r[2 + 3 * k:5 + 3 * k]) for k in range(n)]

    def hidden(self, depth: int) -> np.ndarray:
        return self.debug_read(DBG.SLOT_HIDDEN, depth, np.float32, self.shape.d_model)

    def stage_q(self, stage: int) -> np.ndarray:
        """q (after RoPE) of the token that ran `stage` in the last cycle, at the stage's last layer (SPD_DBG_Q)."""
        return self.debug_read(DBG.Q, stage, np.float32, self.shape.n_q_heads * self.shape.head_dim)

    def stage_att(self, stage: int) -> np.ndarray:
        """The attention output of that layer (SPD_DBG_ATT)."""
        return self.debug_read(DBG.ATT, stage, np.float32, self.shape.n_q_heads * self.shape.head_dim)

    def hfin(self, pos: int) -> np.ndarray:
        return self.debug_read(DBG.HFIN, pos, np.float32, self.shape.d_model)

    def kv_len(self) -> np.ndarray:
        return self.debug_read(DBG.KV_LEN, 0, np.int32, self.shape.n_layers)

    def kv(self, layer: int, which: int, rows: int) -> np.ndarray:
        w = self.shape.n_kv_heads * self.shape.head_dim
        if rows == 0:
            return np.zeros((0, w), dtype=np.uint16)
        return self.debug_read(DBG.KV_V if which else DBG.KV_K, layer, np.uint16, rows * w).reshape(rows, w)

    def cycle_times(self, step_indices) -> np.ndarray:
        """int64[len, 2]: (begin, end) %globaltimer stamps in ns of the cycles with the given step_index values (the
        device keeps the last 1024 cycles; SPD_DBG_CYCLE_TIMES)."""
        ring = self.debug_read(DBG.CYCLE_TIMES, 0, np.uint64, 2 * 1024).reshape(1024, 2).astype(np.int64)
        return ring[(np.asarray(step_indices, dtype=np.int64) - 1) % 1024]

    def phase_profile(self) -> np.ndarray:
        """uint64[160, 168, 6] clock stamps of the last fused cycle (see SPD_DBG_PHASE_PROFILE in spd.h)."""
        return self.debug_read(DBG.PHASE_PROFILE, 0, np.uint64, 160 * 168 * 6).reshape(160, 168, 6)

    def last(self, what: str) -> np.ndarray:
        sel, cnt = {"exit_logits": (DBG.EXIT_LOGITS, self.shape.vocab), "pdm_logits": (DBG.PDM_LOGITS, self.shape.vocab),
                    "pdm_prenorm": (DBG.PDM_PRENORM, self.shape.d_model),
                    "pdm_feat": (DBG.PDM_FEAT, self.shape.d_model * self.shape.n_stages)}[what]
        return self.debug_read(sel, 0, np.float32, cnt)


# ---------------------------------------------------------------------- single operations (device tensors)

def _s(stream):
    return (stream or torch.cuda.current_stream()).cuda_stream


def _chk(rc, name):
    if rc:
        raise SpdError(rc, name)


def op_rmsnorm(x: torch.Tensor, gain: torch.Tensor, eps: float, stream=None) -> torch.Tensor:
    out = torch.empty_like(x)
    _chk(lib().spd_op_rmsnorm(x.data_ptr(), gain.data_ptr(), x.numel(), eps, out.data_ptr(), _s(stream)), "spd_op_rmsnorm")
    return out


def op_gemv(w: torch.Tensor, x: torch.Tensor, stream=None) -> torch.Tensor:
    rows, k = w.shape
    out = torch.empty(rows, dtype=torch.float32, device=x.device)
    _chk(lib().spd_op_gemv(w.data_ptr(), rows, k, x.data_ptr(), out.data_ptr(), _s(stream)), "spd_op_gemv")
    return out


def op_gemm(x: torch.Tensor, w: torch.Tensor, stream=None) -> torch.Tensor:
    """y[M, N] = x[M, K] . w[N, K]^T with the prefill's tcgen05 GEMM (x fp32, w bf16 bits as int16/uint16)."""
    m, k = x.shape
    n = w.shape[0]
    out = torch.empty((m, n), dtype=torch.float32, device=x.device)
    scratch = torch.empty(lib().spd_op_gemm_scratch(m, k), dtype=torch.uint8, device=x.device)
    _chk(lib().spd_op_gemm(x.data_ptr(), w.data_ptr(), m, n, k, out.data_ptr(), scratch.data_ptr(), _s(stream)), "spd_op_gemm")
    return out


def op_rope(vec: torch.Tensor, n_heads: int, head_dim: int, pos: int, base: float, stream=None) -> torch.Tensor:
    out = vec.clone()
    _chk(lib().spd_op_rope(out.data_ptr(), n_heads, head_dim, pos, base, _s(stream)), "spd_op_rope")
    return out


def op_attention(q: torch.Tensor, kc: torch.Tensor, vc: torch.Tensor, t_len: int, n_q_heads: int, n_kv_heads: int,
                 head_dim: int, stream=None) -> torch.Tensor:
    """kc, vc: [n_kv_heads, t_stride, head_dim] 2-byte tensors (head-major cache layout)."""
    t_stride = kc.shape[1]
    out = torch.empty(n_q_heads * head_dim, dtype=torch.float32, device=q.device)
    nbytes = lib().spd_op_attention_scratch(t_len, n_q_heads, head_dim)
    scratch = torch.empty(nbytes // 4 + 1, dtype=torch.float32, device=q.device)
    _chk(lib().spd_op_attention(q.data_ptr(), kc.data_ptr(), vc.data_ptr(), t_len, t_stride, n_q_heads, n_kv_heads,
                                head_dim, out.data_ptr(), scratch.data_ptr(), _s(stream)), "spd_op_attention")
    return out


def op_attention_static(q: torch.Tensor, kc: torch.Tensor, vc: torch.Tensor, t_len: int, n_q_heads: int, n_kv_heads: int,
                        head_dim: int, out: torch.Tensor, stream=None) -> torch.Tensor:
    """spd_op_attention_static: as op_attention, but the library allocates nothing — the caller passes `out`
    (fp32[n_q_heads * head_dim]) and the split partials live in the library's static 2 MiB device array."""
    rc = lib().spd_op_attention_static(q.data_ptr(), kc.data_ptr(), vc.data_ptr(), t_len, kc.shape[1], n_q_heads, n_kv_heads,
                                       head_dim, out.data_ptr(), _s(stream))
    if rc:
        raise SpdError(rc, "spd_op_attention_static")
    return out


def op_silu_mul(gate: torch.Tensor, up: torch.Tensor, stream=None) -> torch.Tensor:
    out = torch.empty_like(gate)
    _chk(lib().spd_op_silu_mul(gate.data_ptr(), up.data_ptr(), gate.numel(), out.data_ptr(), _s(stream)), "spd_op_silu_mul")
    return out


def op_argmax(x: torch.Tensor, stream=None) -> int:
    out = torch.empty(1, dtype=torch.int32, device=x.device)
    _chk(lib().spd_op_argmax(x.data_ptr(), x.numel(), out.data_ptr(), _s(stream)), "spd_op_argmax")
    return int(out.item())


def op_topk_softmax(x: torch.Tensor, top_k: int, temperature: float, use_candidates: bool = True, stream=None):
    """(ids ascending, p) of the filtered distribution of spd_set_sampling."""
    out = torch.zeros(C.sizeof(_Dist), dtype=torch.uint8, device=x.device)
    scratch = torch.empty(lib().spd_op_topk_scratch(), dtype=torch.uint8, device=x.device)
    _chk(lib().spd_op_topk_softmax(x.data_ptr(), x.numel(), top_k, temperature, int(use_candidates), out.data_ptr(),
                                   scratch.data_ptr(), _s(stream)), "spd_op_topk_softmax")
    d = _Dist.from_buffer_copy(out.cpu().numpy().tobytes())
    return _dist_out(d)
