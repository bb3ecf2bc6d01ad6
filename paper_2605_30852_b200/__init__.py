"""B200-native Speculative Pipeline Decoding step (arxiv/paper_2605_30852): thin Python binding over
the C-ABI CUDA library libspd_b200.so (include/spd.h).  Argument marshalling only — every step of the
path runs in the library's kernels.  There is no CPU fallback: importing `binding` raises if the
CUDA library has not been built (python -m paper_2605_30852_b200.build or __graft_entry__.build()).
"""
from .binding import (SPD, StepResult, SpdError, lib, upload_weights, upload_pdm_weights, op_rmsnorm, op_gemv, op_gemm, op_rope,
                      op_attention, op_attention_static, op_silu_mul, op_argmax, op_topk_softmax, DBG, OPT)
from . import reporting

__all__ = ["SPD", "StepResult", "SpdError", "lib", "upload_weights", "upload_pdm_weights", "op_rmsnorm", "op_gemv", "op_gemm", "op_rope",
           "op_attention", "op_attention_static", "op_silu_mul", "op_argmax", "op_topk_softmax", "DBG", "OPT", "reporting"]
