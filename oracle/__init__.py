"""CPU oracle for the SPD step — TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may import
this package.  It shares no code with paper_2605_30852_b200/ (the CUDA path) and neither imports the
other.  `Oracle` is a thin ctypes wrapper over oracle/spd_oracle.c (all arithmetic is in the C file);
`nocache_ref` is a separately written float64 numpy full-sequence model used to pin the C oracle.
"""
from .oracle import Oracle, StepResult, lib, op_rmsnorm, op_gemv, op_rope, op_attention, \
    op_silu_mul, op_argmax, op_f32_to_bf16, op_splitmix64, num_threads, Dist, op_topk_softmax, op_uniform, \
    op_sample_cdf, op_accept, op_sample_residual

__all__ = ["Oracle", "StepResult", "lib", "op_rmsnorm", "op_gemv", "op_rope", "op_attention",
           "op_silu_mul", "op_argmax", "op_f32_to_bf16", "op_splitmix64", "num_threads", "Dist", "op_topk_softmax", "op_uniform", "op_sample_cdf",
           "op_accept", "op_sample_residual"]
