"""Reporting formulas of the paper (no kernels here): PAPER.md:145-156.

alpha = N / K                      step acceptance ratio
S0    = alpha * n                  zero-draft-cost theoretical speedup, Eq. 6
S_adj = S0 * L / (L_s * m + L)     draft-cost-adjusted speedup, Eq. 7, m = k (EAGLE) or n (PPSD)
alpha(p) = 1 / (p + (1 - p) n)     expected alpha when each judged successor is right with prob. p
                                   (a reject costs n cycles, an accept one; derived from PAPER.md:131, :145)
"""
from __future__ import annotations


def alpha(n_tokens: int, n_steps: int) -> float:
    return n_tokens / n_steps


def theoretical_speedup(alpha_: float, n: int) -> float:
    return alpha_ * n


def draft_cost_adjusted(s0: float, n_layers: int, draft_layers: int, serial_draft_steps: int) -> float:
    return s0 * n_layers / (draft_layers * serial_draft_steps + n_layers)


def expected_alpha(p: float, n: int) -> float:
    return 1.0 / (p + (1.0 - p) * n)


def implied_acceptance(alpha_: float, n: int) -> float:
    """Per-token acceptance p implied by a step acceptance ratio: p = (n - 1/alpha) / (n - 1)."""
    return (n - 1.0 / alpha_) / (n - 1.0)


def step_bytes(shape, context_len: int, fill: int | None = None, exited: bool = True, pdm: bool = True) -> dict:
    """Algorithmic HBM bytes of one cycle: every layer's weights of the occupied
    stages once, the touched K/V rows, the tied matrix E once (shared by verify and PDM) and W_p.
    Returns {"strict": layers + KV, "full": strict + E + W_p} in bytes."""
    n = shape.n_stages
    a = n if fill is None else fill
    w_layers = shape.layer_params() * 2 * shape.n_layers * a // n
    kv_row = 2 * shape.n_kv_heads * shape.head_dim * 2
    kv = kv_row * (shape.n_layers * a // n) * context_len
    e = shape.vocab * shape.d_model * 2 if (exited or pdm) else 0
    wp = shape.d_model * n * shape.d_model * 2 if pdm else 0
    return {"strict": w_layers + kv, "full": w_layers + kv + e + wp}
