"""spd_op_attention_static (-m gpu): the allocation-free variant of the split-KV decode attention operation — its split
partials live in a 2 MiB file-scope device array inside the library — against the existing path (spd_op_attention with a
caller-allocated scratch buffer) and against the oracle, on two calls in a row that share the array (a large call, then a
smaller one with other inputs: stale contents of the first must not reach the second).  Named test_zz_* so that pytest
collects it last."""
import numpy as np
import pytest
import torch

import oracle as ora
import spd_inputs as si
from tests._util import rel_err

pytestmark = pytest.mark.gpu
TOL = 2e-5          # tests/test_gpu_ops.py::test_attention


def _dev(a):
    a = np.ascontiguousarray(a)
    if a.dtype == np.uint16:
        return torch.from_numpy(a.view(np.int16)).cuda()
    return torch.from_numpy(a).cuda()


def _case(rng, Hq, Hkv, hd, T):
    q = (rng.standard_normal(Hq * hd) * 2).astype(np.float32)
    K = si.f32_to_bf16_bits((rng.standard_normal((T, Hkv * hd))).astype(np.float32))
    V = si.f32_to_bf16_bits((rng.standard_normal((T, Hkv * hd))).astype(np.float32))
    stride = T + 5
    kc = np.zeros((Hkv, stride, hd), np.uint16)
    vc = np.zeros((Hkv, stride, hd), np.uint16)
    kc[:, :T] = K.reshape(T, Hkv, hd).transpose(1, 0, 2)
    vc[:, :T] = V.reshape(T, Hkv, hd).transpose(1, 0, 2)
    kc[:, T:] = 0x7F80  # +inf beyond T: must never be read
    return q, K, V, _dev(q), _dev(kc), _dev(vc)


def test_static_scratch_attention_matches_the_allocating_path_on_two_calls_in_a_row():
    import paper_2605_30852_b200 as spd
    rng = np.random.default_rng(20260530)
    assert spd.lib().spd_op_attention_static_max_bytes() == 2 << 20
    # call 1: 37 splits x 32 heads (0.6 MB of the array); call 2: 2 splits x 4 heads over the same memory; call 3: call 1's
    # shape again with new inputs
    shapes = [(32, 8, 128, 4609), (4, 2, 64, 130), (32, 8, 128, 2304)]
    for Hq, Hkv, hd, T in [(2, 1, 64, 3), (2, 1, 128, 3)]:   # first launches load the kernels (lazy module loading): not measured
        q, K, V, qd, kcd, vcd = _case(rng, Hq, Hkv, hd, T)
        spd.op_attention_static(qd, kcd, vcd, T, Hq, Hkv, hd, torch.empty(Hq * hd, dtype=torch.float32, device="cuda"))
    for Hq, Hkv, hd, T in shapes:
        q, K, V, qd, kcd, vcd = _case(rng, Hq, Hkv, hd, T)
        want_existing = spd.op_attention(qd, kcd, vcd, T, Hq, Hkv, hd)
        out = torch.full((Hq * hd,), float("nan"), dtype=torch.float32, device="cuda")
        torch.cuda.synchronize()
        free0, alloc0 = torch.cuda.mem_get_info()[0], torch.cuda.memory_allocated()
        spd.op_attention_static(qd, kcd, vcd, T, Hq, Hkv, hd, out)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] >= free0 and torch.cuda.memory_allocated() == alloc0, "the call allocated device memory"
        got = out.cpu().numpy()
        assert np.isfinite(got).all()
        assert rel_err(got, want_existing.cpu().numpy()) < TOL            # the existing path (same arithmetic: in fact identical)
        assert np.array_equal(got, want_existing.cpu().numpy())
        assert rel_err(got, ora.op_attention(q, K, V, Hq, Hkv, hd)) < TOL  # and the oracle


def test_static_scratch_attention_rejects_what_does_not_fit():
    import paper_2605_30852_b200 as spd
    L = spd.lib()
    x = torch.zeros(32 * 128, dtype=torch.float32, device="cuda")
    kv = torch.zeros(16, dtype=torch.int16, device="cuda")
    # 32 heads x head_dim 128: 127 splits need 2 113 280 B > 2 MiB -> SPD_ECAPACITY before any launch; 126 splits fit
    t_big = 127 * 128
    assert L.spd_op_attention_static(x.data_ptr(), kv.data_ptr(), kv.data_ptr(), t_big, t_big, 32, 8, 128, x.data_ptr(), None) == 3
    assert 126 * 32 * 130 * 4 <= L.spd_op_attention_static_max_bytes() < 127 * 32 * 130 * 4
    # argument errors: SPD_EINVAL, nothing launched
    assert L.spd_op_attention_static(None, kv.data_ptr(), kv.data_ptr(), 4, 4, 4, 2, 64, x.data_ptr(), None) == 1
    assert L.spd_op_attention_static(x.data_ptr(), kv.data_ptr(), kv.data_ptr(), 4, 3, 4, 2, 64, x.data_ptr(), None) == 1
    assert L.spd_op_attention_static(x.data_ptr(), kv.data_ptr(), kv.data_ptr(), 4, 4, 4, 3, 64, x.data_ptr(), None) == 1
    assert L.spd_op_attention_static(x.data_ptr(), kv.data_ptr(), kv.data_ptr(), 4, 4, 4, 2, 96, x.data_ptr(), None) == 1
    with pytest.raises(spd.SpdError):
        spd.op_attention_static(x, kv.view(1, 1, 16), kv.view(1, 1, 16), t_big, 32, 8, 128, x)
    torch.cuda.synchronize()
