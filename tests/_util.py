"""Shared helpers for the tests (seeded inputs + cached oracle runs).  No method arithmetic."""
from __future__ import annotations

import functools

import numpy as np

import spd_inputs as si

TINY = si.CONFIGS["tiny"]
# Test-only init: with std 0.02 the tiny model's tied head just echoes the input token (the embedding
# dominates the residual stream), so greedy output is one repeated id.  std 0.08 + random gains makes
# the layers dominate and the tokens diverse, which is what the state-machine pins need.
HOT = dict(std=0.08, random_gains=True)


@functools.lru_cache(maxsize=16)
def weights(name: str = "tiny", n: int | None = None, seed: int = 1234, std: float = 0.08,
            random_gains: bool = True, attention_heavy: bool = False):
    shape = shape_of(name, n)
    return si.make_weights(shape, seed=seed, std=std, random_gains=random_gains,
                           attention_heavy=attention_heavy)


def shape_of(name: str = "tiny", n: int | None = None, **kw):
    shape = si.CONFIGS[name]
    if n is not None:
        shape = shape.replace(n_stages=n)
    if kw:
        shape = shape.replace(**kw)
    return shape


@functools.lru_cache(maxsize=16)
def ar_tokens(name: str = "tiny", n_tokens: int = 64, prompt_seed: int = 1, seed: int = 1234,
              std: float = 0.08, random_gains: bool = True, prompt_len: int | None = None):
    """O-AR greedy tokens [first token from prefill, then n_tokens-1 decode steps]."""
    from oracle import Oracle
    shape = shape_of(name)
    o = Oracle(shape, weights(name, None, seed, std, random_gains), max_seq=4096 if name == "tiny" else None)
    first = o.prefill(si.make_prompt(shape, prompt_seed, prompt_len))
    toks = [first]
    for _ in range(n_tokens - 1):
        toks.append(o.ar_step())
    o.close()
    return tuple(toks)


_LAST = {}


def cached_last(slot: str, key, make):
    """One-entry cache per slot: consecutive test cases that differ only in the engine reuse the seeded inputs (weights of
    the 4B / 9B-class shapes take 10-30 s to generate and ~18 GB on the device) and the oracle's greedy continuation; a new
    key drops the previous entry first."""
    ent = _LAST.get(slot)
    if ent is None or ent[0] != key:
        _LAST.pop(slot, None)
        ent = (key, make())
        _LAST[slot] = ent
    return ent[1]


def rel_err(a: np.ndarray, b: np.ndarray) -> float:
    """SURVEY C-2.18: max_i |a_i - b_i| / max_i |b_i|."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    den = np.max(np.abs(b))
    return float(np.max(np.abs(a - b)) / (den if den > 0 else 1.0))
