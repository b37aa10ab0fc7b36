"""EconoJax CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes loader for ``econojax_oracle.c`` (plain C restatement of the paper's step
rules, see the header for citations and pins).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs import this package.  It imports nothing from ``paper_2410_22165_b200`` and the
product never imports it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "econojax_oracle.c")
_HDR = os.path.join(_HERE, "econojax_oracle.h")
_LIB = os.path.join(_HERE, "liborc.so")

MAX_PRICES, MAX_BRACKETS, MAX_RATE_LEVELS = 16, 16, 32
CRAFT_SINGLE, CRAFT_PER_RESOURCE = 0, 1
SKILL_UNIFORM01, SKILL_PARETO_CLIP, SKILL_NORMAL_CLIP = 0, 1, 2


class OrcParams(C.Structure):
    _fields_ = [
        ("num_prices", C.c_int32), ("prices", C.c_int32 * MAX_PRICES),
        ("episode_length", C.c_int32), ("tax_period", C.c_int32),
        ("num_brackets", C.c_int32), ("thresholds", C.c_float * MAX_BRACKETS),
        ("num_rate_levels", C.c_int32), ("rate_table", C.c_float * MAX_RATE_LEVELS),
        ("allow_noop", C.c_int32), ("starting_coin", C.c_float), ("order_expiry", C.c_int32),
        ("max_active_orders", C.c_int32), ("book_cap", C.c_int32),
        ("craft_units", C.c_int32), ("craft_distinct", C.c_int32), ("craft_mode", C.c_int32),
        ("labor_craft", C.c_float), ("labor_gather", C.c_float), ("labor_trade", C.c_float),
        ("eta", C.c_float), ("omega", C.c_float), ("craft_scale", C.c_float),
        ("taxes_enabled", C.c_int32), ("skill_init", C.c_int32),
        ("skill_clip_lo", C.c_float), ("skill_clip_hi", C.c_float),
        ("obs_scale_coin", C.c_float), ("obs_scale_count", C.c_float),
        ("obs_scale_price", C.c_float), ("obs_scale_labor", C.c_float),
        ("env_id_base", C.c_uint32),
        ("skill_growth_rate", C.c_float), ("skill_max", C.c_float),
        ("skill_mean", C.c_float), ("skill_std", C.c_float),
    ]


class OrcOrder(C.Structure):
    _fields_ = [("price", C.c_int32), ("owner", C.c_int32), ("placed_at", C.c_int32), ("key", C.c_uint32)]


class OrcTrade(C.Structure):
    _fields_ = [("buyer", C.c_int32), ("seller", C.c_int32), ("bid_price", C.c_int32),
                ("ask_price", C.c_int32), ("price", C.c_int32)]


def build(force: bool = False) -> str:
    """Compile the oracle with contraction off (G31). Returns the path of the library."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
                               "-Wall", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None
_lock = threading.Lock()


def lib():
    global _lib
    with _lock:
        if _lib is None:
            L = C.CDLL(build())
            u32p, i32p, f32p = C.POINTER(C.c_uint32), C.POINTER(C.c_int32), C.POINTER(C.c_float)
            L.orc_philox4x32_10.argtypes = [u32p, u32p, u32p]
            L.orc_u01.argtypes = [C.c_uint32]; L.orc_u01.restype = C.c_float
            L.orc_gather_amount.argtypes = [C.c_float, C.c_float]; L.orc_gather_amount.restype = C.c_int32
            L.orc_num_actions.argtypes = [C.c_int32] * 4; L.orc_num_actions.restype = C.c_int32
            L.orc_craft_consume.argtypes = [i32p] + [C.c_int32] * 5; L.orc_craft_consume.restype = C.c_int32
            L.orc_marginal_tax.argtypes = [C.c_float, f32p, f32p, C.c_int32]; L.orc_marginal_tax.restype = C.c_float
            L.orc_utility.argtypes = [C.c_double] * 3; L.orc_utility.restype = C.c_double
            L.orc_gini.argtypes = [f32p, C.c_int32]; L.orc_gini.restype = C.c_double
            dp = C.POINTER(C.c_double)
            L.orc_social_welfare.argtypes = [f32p, C.c_int32, C.c_double, dp, dp, dp]
            L.orc_stats.argtypes = [f32p, C.c_int32, dp, dp, f32p]
            L.orc_match_book.argtypes = [C.POINTER(OrcOrder), i32p, C.POINTER(OrcOrder), i32p, C.POINTER(OrcTrade), C.c_int32]
            L.orc_match_book.restype = C.c_int32
            L.orc_create.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.POINTER(OrcParams)]; L.orc_create.restype = C.c_void_p
            L.orc_destroy.argtypes = [C.c_void_p]
            L.orc_last_error.restype = C.c_char_p
            L.orc_obs_dim_pop.argtypes = [C.c_void_p]; L.orc_obs_dim_pop.restype = C.c_int32
            L.orc_obs_dim_gov.argtypes = [C.c_void_p]; L.orc_obs_dim_gov.restype = C.c_int32
            L.orc_reset.argtypes = [C.c_void_p, C.c_uint64]
            L.orc_begin_episode.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32]
            L.orc_step_auto.argtypes = [C.c_void_p, C.c_int32, C.c_int32] + [C.c_void_p] * 6
            L.orc_observe.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
            L.orc_step.argtypes = [C.c_void_p, C.c_int32, C.c_int32] + [C.c_void_p] * 6
            L.orc_draw_actions.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
            L.orc_action_mask.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p]
            L.orc_draw_actions_masked.argtypes = L.orc_draw_actions.argtypes
            L.orc_state_words.argtypes = [C.c_void_p]; L.orc_state_words.restype = C.c_size_t
            L.orc_get_state.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p]
            L.orc_set_agent.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_float, i32p, f32p, C.c_float]
            L.orc_set_rates.argtypes = [C.c_void_p, C.c_int32, f32p]
            L.orc_get_agent_f.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32]; L.orc_get_agent_f.restype = C.c_float
            _lib = L
    return _lib


def make_params(d: dict) -> OrcParams:
    """Fill the oracle's own parameter struct from a plain dict (see inputs.default_params)."""
    p = OrcParams()
    prices = list(d["prices"])
    p.num_prices = len(prices)
    for i, v in enumerate(prices):
        p.prices[i] = int(v)
    thr = list(d["thresholds"])
    p.num_brackets = len(thr) + 1
    for i, v in enumerate(thr):
        p.thresholds[i] = float(v)
    table = list(d["rate_table"])
    p.num_rate_levels = len(table)
    for i, v in enumerate(table):
        p.rate_table[i] = float(v)
    for name in ("episode_length", "tax_period", "allow_noop", "order_expiry", "max_active_orders", "book_cap",
                 "craft_units", "craft_distinct", "craft_mode", "taxes_enabled", "skill_init", "env_id_base"):
        setattr(p, name, int(d[name]))
    for name in ("starting_coin", "labor_craft", "labor_gather", "labor_trade", "eta", "omega", "craft_scale",
                 "skill_clip_lo", "skill_clip_hi", "obs_scale_coin", "obs_scale_count", "obs_scale_price",
                 "obs_scale_labor", "skill_growth_rate", "skill_max", "skill_mean", "skill_std"):
        setattr(p, name, float(d[name]))
    return p


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class OracleEnv:
    """E independent economies stepped one after another by the C oracle."""

    def __init__(self, E: int, N: int, R: int, params: dict):
        self.L = lib()
        self.E, self.N, self.R = E, N, R
        self.params = dict(params)
        self._p = make_params(params)
        self.h = self.L.orc_create(E, N, R, C.byref(self._p))
        if not self.h:
            raise ValueError("orc_create: bad field %s" % self.L.orc_last_error().decode())
        self.B = self._p.num_brackets
        self.D_pop = self.L.orc_obs_dim_pop(self.h)
        self.D_gov = self.L.orc_obs_dim_gov(self.h)
        self.A = self.L.orc_num_actions(R, self._p.num_prices, self._p.craft_mode, self._p.allow_noop)
        self.state_words = int(self.L.orc_state_words(self.h))

    def __del__(self):
        if getattr(self, "h", None):
            self.L.orc_destroy(self.h)
            self.h = None

    def reset(self, seed: int):
        self.L.orc_reset(self.h, C.c_uint64(seed))

    def observe(self, env_begin=0, env_count=None):
        n = self.E - env_begin if env_count is None else env_count
        obs_pop = np.zeros((n, self.N, self.D_pop), np.float32)
        obs_gov = np.zeros((n, self.D_gov), np.float32)
        self.L.orc_observe(self.h, env_begin, n, _ptr(obs_pop), _ptr(obs_gov))
        return obs_pop, obs_gov

    def begin_episode(self, episode: int, env_begin=0, env_count=None):
        """f4: start episode `episode` in the given envs (orc_reset starts episode 0 everywhere)."""
        n = self.E - env_begin if env_count is None else env_count
        self.L.orc_begin_episode(self.h, env_begin, n, int(episode))

    def step(self, actions, gov_actions, env_begin=0, want_obs=True, auto_reset=False):
        actions = np.ascontiguousarray(actions, np.int32)
        gov_actions = np.ascontiguousarray(gov_actions, np.int32)
        n = actions.shape[0]
        assert actions.shape == (n, self.N) and gov_actions.shape == (n, self.B)
        obs_pop = np.zeros((n, self.N, self.D_pop), np.float32) if want_obs else None
        obs_gov = np.zeros((n, self.D_gov), np.float32) if want_obs else None
        rew = np.zeros((n, self.N + 1), np.float32)
        done = np.zeros((n,), np.uint8)
        fn = self.L.orc_step_auto if auto_reset else self.L.orc_step
        fn(self.h, env_begin, n, _ptr(actions), _ptr(gov_actions), _ptr(obs_pop), _ptr(obs_gov), _ptr(rew), _ptr(done))
        return obs_pop, obs_gov, rew, done

    def draw_actions(self, cdf, env_begin=0, env_count=None, masked=False):
        """Rollout-mode generator (G30); masked=True: restricted to the available actions (f1)."""
        n = self.E - env_begin if env_count is None else env_count
        cdf = np.ascontiguousarray(cdf, np.uint32)
        assert cdf.shape == (self.A,)
        actions = np.zeros((n, self.N), np.int32)
        gov = np.zeros((n, self.B), np.int32)
        fn = self.L.orc_draw_actions_masked if masked else self.L.orc_draw_actions
        fn(self.h, env_begin, n, _ptr(cdf), _ptr(actions), _ptr(gov))
        return actions, gov

    def action_mask(self, env_begin=0, env_count=None):
        """[n][N][A] uint8, 1 = action available in the current state (f1)."""
        n = self.E - env_begin if env_count is None else env_count
        m = np.zeros((n, self.N, self.A), np.uint8)
        self.L.orc_action_mask(self.h, env_begin, n, _ptr(m))
        return m

    def get_state(self, env_begin=0, env_count=None):
        n = self.E - env_begin if env_count is None else env_count
        w = np.zeros((n, self.state_words), np.int32)
        self.L.orc_get_state(self.h, env_begin, n, _ptr(w))
        return w

    def set_agent(self, env, agent, coin, inv=None, SG=None, SC=0.0):
        i32p, f32p = C.POINTER(C.c_int32), C.POINTER(C.c_float)
        inv_a = None if inv is None else (C.c_int32 * self.R)(*[int(v) for v in inv])
        sg_a = None if SG is None else (C.c_float * self.R)(*[float(v) for v in SG])
        self.L.orc_set_agent(self.h, env, agent, float(coin),
                             C.cast(inv_a, i32p) if inv_a is not None else None,
                             C.cast(sg_a, f32p) if sg_a is not None else None, float(SC))

    def set_rates(self, env, rates):
        arr = (C.c_float * MAX_BRACKETS)(*[float(v) for v in rates])
        self.L.orc_set_rates(self.h, env, C.cast(arr, C.POINTER(C.c_float)))

    def agent_f(self, env, agent, what):
        return float(self.L.orc_get_agent_f(self.h, env, agent, {"coin": 0, "labor": 1, "income": 2}[what]))


def parse_state(words: np.ndarray) -> dict:
    """Split one env's canonical dump into named arrays."""
    w = np.asarray(words, np.int32)
    t, N, R, B, P, cap = (int(v) for v in w[:6])
    out = {"t": t, "N": N, "R": R, "B": B, "P": P, "cap": cap,
           "counters": w[6:11].copy(), "u_g_prev": float(w[11:13].view(np.float64)[0])}
    q = 13
    out["rates"] = w[q:q + B].view(np.float32).copy(); q += B
    out["last_price"] = w[q:q + R].copy(); q += R
    rec = 6 + 3 * R
    ag = w[q:q + N * rec].reshape(N, rec); q += N * rec
    out["coin"] = ag[:, 0].copy().view(np.float32)
    out["esc_coin"] = ag[:, 1].copy()
    out["SC"] = ag[:, 2].copy().view(np.float32)
    out["labor"] = ag[:, 3].copy().view(np.float32)
    out["income"] = ag[:, 4].copy().view(np.float32)
    out["n_live"] = ag[:, 5].copy()
    out["inv"] = ag[:, 6:6 + R].copy()
    out["esc_res"] = ag[:, 6 + R:6 + 2 * R].copy()
    out["SG"] = ag[:, 6 + 2 * R:6 + 3 * R].copy().view(np.float32)
    books = []
    for _ in range(2 * R):
        n = int(w[q]); q += 1
        books.append(w[q:q + 3 * n].reshape(n, 3).copy())
        q += 3 * cap
    out["books"] = books  # index 2*r + side, rows (price, owner, placed_at) in priority order
    out["episode"] = int(w[q]) if q < len(w) else 0  # f4: last word
    return out
