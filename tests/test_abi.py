"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/spd.h declares,
validates configurations on the host, and refuses to run without a GPU (no CPU fallback)."""
import ctypes as C
import os
import re

import pytest
import torch

import spd_inputs as si

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2605_30852_b200 import build
    build.build()
    from paper_2605_30852_b200 import binding
    return binding.lib()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "spd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(spd_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lib):
    syms = declared_symbols()
    assert {"spd_create", "spd_prefill", "spd_step", "spd_rollback", "spd_query_sizes", "spd_destroy",
            "spd_step_many", "spd_set_forced", "spd_debug_read", "spd_last_error", "spd_set_sampling",
            "spd_op_topk_softmax"} <= set(syms)
    for s in syms:
        assert hasattr(lib, s), s


def test_sample_record_layout_matches_the_header(lib):
    """The binding's ctypes mirror of spd_sample_record / spd_sample_dist has the header's field order and size."""
    from paper_2605_30852_b200.binding import _Dist, _SampleRec, MAX_TOPK
    text = open(os.path.join(ROOT, "include", "spd.h")).read()
    assert int(re.search(r"#define SPD_MAX_TOPK (\d+)", text).group(1)) == MAX_TOPK == 64
    assert C.sizeof(_Dist) == 4 + 8 * MAX_TOPK and C.sizeof(_SampleRec) == 2 * C.sizeof(_Dist) + 32
    body = re.search(r"typedef struct \{([^}]*)\} spd_sample_record;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = re.findall(r"\b([a-z_]+)\s*[,;]", body)
    assert names == [k for k, _ in _SampleRec._fields_]


def test_query_sizes_and_validation(lib):
    from paper_2605_30852_b200.binding import query_sizes, SpdError
    for name, shape in si.CONFIGS.items():
        repack, kv, work = query_sizes(shape)
        assert kv == shape.n_layers * 2 * shape.n_kv_heads * shape.head_dim * 2 * shape.max_seq
        assert work > shape.max_seq * shape.d_model * 4 and repack >= 256
    tiny = si.CONFIGS["tiny"]
    for bad in (tiny.replace(n_stages=3), tiny.replace(n_q_heads=3), tiny.replace(head_dim=63),
                tiny.replace(d_model=260), tiny.replace(n_stages=0), tiny.replace(vocab=1)):
        with pytest.raises(SpdError) as e:
            query_sizes(bad)
        assert e.value.status == 1  # SPD_EINVAL


def test_pdm_query_sizes_and_validation(lib):
    """spd_pdm_query_sizes needs no GPU: the PDM's cache is L_s layers of the target's per-layer cache, the work buffer
    holds at least the anchors H^b of every position ([max_seq][m][d] fp32, m = 5 anchors for L >= 8)."""
    from paper_2605_30852_b200.binding import _PdmSizes, _cfg_of
    for name in ("tiny", "9b_n4"):
        shape = si.CONFIGS[name]
        cfg = _cfg_of(shape, shape.max_seq, 0)
        sz = _PdmSizes()
        assert lib.spd_pdm_query_sizes(C.byref(cfg), 3, 300, C.byref(sz)) == 0
        assert sz.kv_bytes == 3 * 2 * shape.n_kv_heads * shape.head_dim * 2 * shape.max_seq
        assert sz.work_bytes > shape.max_seq * si.pdm_anchor_count(shape.n_layers) * shape.d_model * 4
        for layers, vocab in ((0, 300), (3, 0), (3, shape.vocab + 1), (1000, 300)):
            assert lib.spd_pdm_query_sizes(C.byref(cfg), layers, vocab, C.byref(sz)) == 1      # SPD_EINVAL
    assert lib.spd_pdm_attach(None, None, None, None) == 1
    assert si.pdm_anchor_count(32) == 5 and si.pdm_anchor_count(8) == 5 and si.pdm_anchor_count(4) == 4


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_gpu_means_no_compute_not_a_fallback(lib):
    from paper_2605_30852_b200.binding import _Cfg, _Weights, _Buffers, _cfg_of
    tiny = si.CONFIGS["tiny"]
    cfg = _cfg_of(tiny, tiny.max_seq, 0)
    dummy = (C.c_void_p * tiny.n_layers)(*[8] * tiny.n_layers)
    w = _Weights()
    for k, _ in _Weights._fields_:
        setattr(w, k, C.cast(dummy, C.POINTER(C.c_void_p)) if k not in ("embed", "final_norm", "pdm_proj", "pdm_norm") else 8)
    bufs = _Buffers(8, 8, 8, None, None, 1 << 40, 1 << 40, 1 << 40)
    h = C.c_void_p()
    assert lib.spd_create(C.byref(cfg), C.byref(w), C.byref(bufs), C.byref(h)) == 4  # SPD_ECUDA
    assert not h.value
    assert lib.spd_step(None, None) == 1 and lib.spd_destroy(None) == 1
    assert lib.spd_set_sampling(None, 1.0, 50, 1) == 1                       # SPD_EINVAL: null ctx
    assert lib.spd_op_topk_softmax(None, 8, 4, 1.0, 1, None, None, None) == 1
    assert lib.spd_op_topk_scratch() >= 2 * 2048 * 4
    assert b"null" in lib.spd_last_error(None)


def test_reporting_formulas_match_the_papers_tables():
    from paper_2605_30852_b200 import reporting as R
    gold = os.path.join(ROOT, "tests", "golden")
    for line in open(os.path.join(gold, "paper_table4.txt")):
        if line.startswith("#") or not line.strip():
            continue
        n, L, Ls, s0, sadj = line.split()
        got = R.draft_cost_adjusted(float(s0), int(L), int(Ls), int(n))      # Eq. 7 (PPSD form: m = n)
        assert abs(got - float(sadj)) < 0.011, line
    for line in open(os.path.join(gold, "paper_table2_alpha.txt")):
        if line.startswith("#") or not line.strip():
            continue
        _, n, s0 = line.split()
        n, s0 = int(n), float(s0)
        a = s0 / n
        assert abs(R.theoretical_speedup(a, n) - s0) < 1e-12                  # Eq. 6
        p = R.implied_acceptance(a, n)
        assert 0.6 < p < 0.92                                                  # BASELINE.md's quoted range
        assert abs(R.expected_alpha(p, n) - a) < 1e-12                        # the two forms are inverses
    assert R.expected_alpha(1.0, 4) == 1.0 and abs(R.expected_alpha(0.6, 4) - 1 / 2.2) < 1e-12
    b = R.step_bytes(si.CONFIGS["9b_n4"], 2176)
    assert abs(b["strict"] / 1e9 - 12.634) < 0.01 and abs(b["full"] / 1e9 - 14.013) < 0.01
