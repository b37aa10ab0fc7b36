"""Oracle of step a12 (policy forward + sampling) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain numpy, binary64.  What it follows:

* the paper fixes the network shape only: two hidden layers of 128 tanh units (P:240,
  Table 2) with a categorical head; BASELINE.json configs[4] fixes bf16
  weights ~ N(0, 0.02) and "categorical action sampling via Philox keyed by (seed, env, agent,
  step)";
* DESIGN.md reading G33 fixes the arithmetic: observations and activations are rounded to
  bfloat16 (nearest even) before each layer, products are accumulated in higher precision
  (here binary64), tanh between layers, logits = last affine map; the action of a head is the
  first index a with u < sum_{j<=a} softmax(l)_j, u = (x >> 8) * 2^-24 from the Philox word of
  G30 (population: stream 0 word 0; government head b: stream 1 + b // 4, word b % 4).

Pins (tests/test_oracle_policy.py): a hand-computed 1-2-2-2 network, bf16 rounding against
hand values and torch's bfloat16 cast, the whole forward against torch.nn.functional.linear,
softmax/CDF special cases (uniform logits -> floor(u A); one dominant logit), brute-force
interval membership.  Shares no code with the CUDA path.
"""
from __future__ import annotations

import ctypes as C

import numpy as np


def bf16_round(x) -> np.ndarray:
    """Nearest-even rounding of binary64 values to bfloat16, returned as binary64."""
    x = np.asarray(x, np.float64)
    out = np.zeros_like(x)
    nz = (x != 0) & np.isfinite(x)
    m, e = np.frexp(x[nz])              # x = m * 2^e, 0.5 <= |m| < 1
    q = np.rint(m * 256.0)              # 8 significant bits; np.rint rounds half to even
    out[nz] = np.ldexp(q, e - 8)
    out[~np.isfinite(x)] = x[~np.isfinite(x)]
    return out


def bf16_bits_to_f64(bits) -> np.ndarray:
    """uint16 bfloat16 bit patterns -> binary64 values."""
    b = np.asarray(bits, np.uint16).astype(np.uint32) << 16
    return b.view(np.float32).astype(np.float64)


def mlp_logits(net: dict, obs_rows) -> np.ndarray:
    """logits [rows][out] of the tanh MLP `net` (keys w1,w2,w3: bf16 bits [out][in]; b1,b2,b3: f32)."""
    x = bf16_round(np.asarray(obs_rows, np.float32).astype(np.float64))
    w1, w2, w3 = (bf16_bits_to_f64(net[k]) for k in ("w1", "w2", "w3"))
    b1, b2, b3 = (np.asarray(net[k], np.float32).astype(np.float64) for k in ("b1", "b2", "b3"))
    h1 = bf16_round(np.tanh(x @ w1.T + b1))
    h2 = bf16_round(np.tanh(h1 @ w2.T + b2))
    return h2 @ w3.T + b3


def softmax_cdf(logits_head, mask=None) -> np.ndarray:
    """Cumulative softmax probabilities of one head (binary64), 1 from the last available entry on.
    mask (f1): actions with mask == 0 get probability exactly 0 -- they are left out
    of the maximum and of the normalising sum, i.e. their logit is -inf."""
    l = np.asarray(logits_head, np.float64)
    ok = np.ones(l.shape, bool) if mask is None else np.asarray(mask).astype(bool)
    p = np.where(ok, np.exp(l - l[ok].max()), 0.0)
    c = np.cumsum(p / p.sum())
    c[np.flatnonzero(ok)[-1]:] = 1.0
    return c


def sample(logits_head, u: float, mask=None) -> int:
    """First index a with u < CDF[a] (G33); an unavailable action has an empty interval."""
    return int(np.searchsorted(softmax_cdf(logits_head, mask), u, side="right"))


def sample_consistent(logits_head, u: float, action: int, eps: float, mask=None) -> bool:
    """True if `action` is what `sample` returns for some u' within eps of u: u lies in the action's
    CDF interval widened by eps (the teacher-forced acceptance test of G33).  Under a mask an
    unavailable action is never consistent."""
    if mask is not None and not mask[action]:
        return False
    c = softmax_cdf(logits_head, mask)
    lo = 0.0 if action == 0 else c[action - 1]
    return bool(lo - eps <= u < c[action] + eps)


def philox_u(seed: int, env: int, agent: int, t: int, stream: int, word: int) -> float:
    """u = (x >> 8) * 2^-24 of the counter-based generator of G30 (the C oracle's Philox)."""
    from . import lib

    L = lib()
    ctr = (C.c_uint32 * 4)(env & 0xFFFFFFFF, agent, t, stream)
    key = (C.c_uint32 * 2)(seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF)
    out = (C.c_uint32 * 4)()
    L.orc_philox4x32_10(ctr, key, out)
    return float(out[word] >> 8) * (1.0 / 16777216.0)
