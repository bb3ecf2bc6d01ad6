"""Seeded synthetic inputs for the SPD hot path (weights, prompts, KV filler).

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA path
(`paper_2605_30852_b200/`).  It holds none of the method's arithmetic: it only draws
random numbers and names the model shapes of BASELINE.json `configs`.  Both sides receive
the very same bytes; neither regenerates them.

Recipe: every matrix is bf16, N(0, 0.02) drawn in float32 by a
counter-based Box-Muller generator keyed by (seed, tensor id, layer) (spd_inputs/fastgen.c) and
rounded to bf16 with round-to-nearest-even;
norm gains are 1.0 (or, for the test-only variant, U[0.5, 1.5] rounded to bf16); prompt token
ids are uniform on [0, vocab).
"""
from .gen import (CONFIGS, ModelShape, make_weights, make_prompt, f32_to_bf16_bits,
                  bf16_bits_to_f32, layer_tensor_names, make_kv_filler, make_tensor, shapes_of, make_echo,
                  make_pdm_weights, pdm_anchor_count)

__all__ = ["CONFIGS", "ModelShape", "make_weights", "make_prompt", "f32_to_bf16_bits",
           "bf16_bits_to_f32", "layer_tensor_names", "make_kv_filler", "make_tensor", "shapes_of", "make_echo",
           "make_pdm_weights", "pdm_anchor_count"]
