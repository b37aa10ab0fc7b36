"""Thin ctypes binding of ``include/econojax.h`` -- argument marshalling only.

Every function below has the name and the arguments of the C entry point it calls; pointers
are passed as integers (``tensor.data_ptr()`` for device memory owned by PyTorch,
``ndarray.ctypes.data`` for host memory).  ``Env`` is a small convenience wrapper that owns
the handle and allocates the PyTorch tensors.  There is no CPU fallback: if the CUDA library
is missing, ``lib()`` raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

MAX_PRICES, MAX_BRACKETS, MAX_RATE_LEVELS = 16, 16, 32
EJ_OK, EJ_ERR_PARAM, EJ_ERR_NOMEM, EJ_ERR_CUDA, EJ_ERR_STATE = 0, -1, -2, -3, -4


class EjParams(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32),
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


class EjLayoutInfo(C.Structure):
    _fields_ = [
        ("E", C.c_int32), ("N", C.c_int32), ("R", C.c_int32), ("P", C.c_int32), ("B", C.c_int32), ("L", C.c_int32),
        ("A", C.c_int32), ("base_craft", C.c_int32), ("base_buy", C.c_int32), ("base_sell", C.c_int32),
        ("noop_action", C.c_int32), ("D_pop", C.c_int32), ("D_gov", C.c_int32), ("D_gov_pad", C.c_int32),
        ("gov_obs_offset", C.c_size_t), ("obs_floats", C.c_size_t), ("rew_floats", C.c_size_t),
        ("state_words", C.c_size_t), ("device_state_bytes", C.c_size_t), ("smem_bytes", C.c_size_t),
        ("threads_per_env", C.c_int32), ("D_priv", C.c_int32), ("D_shared", C.c_int32), ("D_shared_pad", C.c_int32),
    ]


class EjRolloutIO(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("ring_depth", C.c_int32),
        ("actions_in", C.c_void_p), ("gov_actions_in", C.c_void_p),
        ("obs_ring", C.c_void_p), ("rew_ring", C.c_void_p), ("done_ring", C.c_void_p),
        ("actions_ring", C.c_void_p), ("gov_actions_ring", C.c_void_p),
        ("pop_logits_ring", C.c_void_p), ("gov_logits_ring", C.c_void_p),
        ("obs_priv_ring", C.c_void_p), ("obs_shared_ring", C.c_void_p), ("obs_gov_ring", C.c_void_p),
        ("auto_reset", C.c_int32), ("reserved0", C.c_int32),
    ]


class EjMlp(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("in_dim", C.c_int32), ("hidden", C.c_int32), ("out_dim", C.c_int32),
        ("w1", C.c_void_p), ("w2", C.c_void_p), ("w3", C.c_void_p),
        ("b1", C.c_void_p), ("b2", C.c_void_p), ("b3", C.c_void_p),
    ]


EXPORTS = ("ej_create", "ej_destroy", "ej_set_stream", "ej_layout", "ej_last_error", "ej_reset", "ej_observe",
           "ej_step", "ej_step_host", "ej_step_host_factored", "ej_rollout", "ej_set_action_cdf", "ej_get_state", "ej_set_state",
           "ej_launch_count", "ej_set_policy", "ej_policy_act", "ej_action_mask", "ej_set_action_masking", "ej_rollout_noalloc")
NOALLOC_SCRATCH_BYTES = 4 << 20

_lib = None


def lib():
    """Load libeconojax.so (building it in-tree if the source is newer).  Raises if unavailable."""
    global _lib
    if _lib is None:
        path = os.environ.get("EJ_LIB")  # a prebuilt library (development builds); default: the in-tree build
        if not path:
            path = _build.LIB
            if not os.path.exists(path) or os.path.getmtime(path) < os.path.getmtime(_build.SRC):
                path = _build.build_lib()
        L = C.CDLL(path)
        vp = C.c_void_p
        L.ej_create.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.POINTER(EjParams), C.POINTER(vp)]
        L.ej_destroy.argtypes = [vp]
        L.ej_set_stream.argtypes = [vp, vp]
        L.ej_layout.argtypes = [vp, C.POINTER(EjLayoutInfo)]
        L.ej_last_error.argtypes = [vp]; L.ej_last_error.restype = C.c_char_p
        L.ej_reset.argtypes = [vp, C.c_uint64]
        L.ej_observe.argtypes = [vp, vp]
        L.ej_action_mask.argtypes = [vp, vp]
        L.ej_set_action_masking.argtypes = [vp, C.c_int32]
        L.ej_step.argtypes = [vp, vp, vp, vp, vp, vp]
        L.ej_step_host.argtypes = [vp, vp, vp, vp, vp, vp]
        L.ej_step_host_factored.argtypes = [vp] * 8
        L.ej_rollout.argtypes = [vp, C.c_int32, C.POINTER(EjRolloutIO)]
        L.ej_set_action_cdf.argtypes = [vp, vp, C.c_int32]
        L.ej_get_state.argtypes = [vp, C.c_int32, C.c_int32, vp, C.c_size_t]
        L.ej_set_state.argtypes = [vp, C.c_int32, C.c_int32, vp, C.c_size_t]
        L.ej_launch_count.argtypes = [vp]; L.ej_launch_count.restype = C.c_int64
        L.ej_set_policy.argtypes = [vp, C.POINTER(EjMlp), C.POINTER(EjMlp)]
        L.ej_policy_act.argtypes = [vp, vp, vp, vp, vp, vp]
        L.ej_rollout_noalloc.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.POINTER(EjParams), C.c_uint64, C.c_int32, vp, vp, vp, vp, vp, vp]
        for name in EXPORTS:
            if name not in ("ej_last_error", "ej_launch_count"):
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


class EjError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("econojax error %d: %s" % (code, msg))
        self.code = code


def make_params(d: dict) -> EjParams:
    """Fill ej_params from a plain dict (see inputs.default_params)."""
    p = EjParams()
    p.struct_size = C.sizeof(EjParams)
    prices = list(d["prices"])
    p.num_prices = len(prices)
    for i, v in enumerate(prices[:MAX_PRICES]):
        p.prices[i] = int(v)
    thr = list(d["thresholds"])
    p.num_brackets = len(thr) + 1
    for i, v in enumerate(thr[:MAX_BRACKETS]):
        p.thresholds[i] = float(v)
    table = list(d["rate_table"])
    p.num_rate_levels = len(table)
    for i, v in enumerate(table[:MAX_RATE_LEVELS]):
        p.rate_table[i] = float(v)
    for name in ("episode_length", "tax_period", "allow_noop", "order_expiry", "max_active_orders", "book_cap",
                 "craft_units", "craft_distinct", "craft_mode", "taxes_enabled", "skill_init", "env_id_base"):
        setattr(p, name, int(d[name]))
    for name in ("starting_coin", "labor_craft", "labor_gather", "labor_trade", "eta", "omega", "craft_scale",
                 "skill_clip_lo", "skill_clip_hi", "obs_scale_coin", "obs_scale_count", "obs_scale_price",
                 "obs_scale_labor", "skill_growth_rate", "skill_max", "skill_mean", "skill_std"):
        setattr(p, name, float(d[name]))
    return p


def _check(h, rc):
    if rc != EJ_OK:
        raise EjError(rc, (lib().ej_last_error(h) or b"").decode())


# ---- same-name wrappers: marshalling only ----
def ej_create(E, N, R, params: EjParams):
    h = C.c_void_p()
    rc = lib().ej_create(E, N, R, C.byref(params), C.byref(h))
    _check(None, rc)
    return h


def ej_destroy(h):
    _check(h, lib().ej_destroy(h))


def ej_set_stream(h, cuda_stream: int):
    _check(h, lib().ej_set_stream(h, cuda_stream))


def ej_layout(h) -> EjLayoutInfo:
    info = EjLayoutInfo()
    _check(h, lib().ej_layout(h, C.byref(info)))
    return info


def ej_last_error(h) -> str:
    return (lib().ej_last_error(h) or b"").decode()


def ej_reset(h, seed: int):
    _check(h, lib().ej_reset(h, C.c_uint64(seed)))


def ej_observe(h, obs_out: int):
    _check(h, lib().ej_observe(h, obs_out))


def ej_set_action_masking(h, on: bool):
    _check(h, lib().ej_set_action_masking(h, 1 if on else 0))


def ej_action_mask(h, mask_out: int):
    _check(h, lib().ej_action_mask(h, mask_out))


def ej_step(h, actions: int, gov_actions: int, obs_out: int | None, rew_out: int | None, done_out: int | None):
    _check(h, lib().ej_step(h, actions, gov_actions, obs_out, rew_out, done_out))


def ej_step_host(h, actions: int, gov_actions: int, obs_out: int | None, rew_out: int | None, done_out: int | None):
    _check(h, lib().ej_step_host(h, actions, gov_actions, obs_out, rew_out, done_out))


def ej_step_host_factored(h, actions: int, gov_actions: int, priv_out: int, shared_out: int, gov_obs_out: int | None,
                          rew_out: int | None, done_out: int | None):
    _check(h, lib().ej_step_host_factored(h, actions, gov_actions, priv_out, shared_out, gov_obs_out, rew_out, done_out))


def ej_rollout(h, T: int, io: EjRolloutIO | None):
    _check(h, lib().ej_rollout(h, T, C.byref(io) if io is not None else None))


def ej_set_action_cdf(h, cdf: int, A: int):
    _check(h, lib().ej_set_action_cdf(h, cdf, A))


def ej_get_state(h, env_begin: int, env_count: int, words: int, n_words: int):
    _check(h, lib().ej_get_state(h, env_begin, env_count, words, n_words))


def ej_set_state(h, env_begin: int, env_count: int, words: int, n_words: int):
    _check(h, lib().ej_set_state(h, env_begin, env_count, words, n_words))


def ej_set_policy(h, pop: EjMlp | None, gov: EjMlp | None):
    _check(h, lib().ej_set_policy(h, C.byref(pop) if pop is not None else None, C.byref(gov) if gov is not None else None))


def ej_policy_act(h, obs: int, actions_out: int, gov_actions_out: int, pop_logits_out: int | None, gov_logits_out: int | None):
    _check(h, lib().ej_policy_act(h, obs, actions_out, gov_actions_out, pop_logits_out, gov_logits_out))


def make_mlp(net: dict) -> EjMlp:
    """ej_mlp over host arrays: net = {"w1","w2","w3": uint16 bf16 bits [out][in]; "b1","b2","b3": float32}.
    The arrays must stay alive until ej_set_policy returns (the struct keeps them referenced)."""
    m = EjMlp()
    m.struct_size = C.sizeof(EjMlp)
    keep = []
    for k in ("w1", "w2", "w3"):
        a = np.ascontiguousarray(net[k], np.uint16)
        keep.append(a)
        setattr(m, k, a.ctypes.data)
    for k in ("b1", "b2", "b3"):
        a = np.ascontiguousarray(net[k], np.float32)
        keep.append(a)
        setattr(m, k, a.ctypes.data)
    m.in_dim, m.hidden, m.out_dim = keep[0].shape[1], keep[0].shape[0], keep[2].shape[0]
    m._keep = keep
    return m


def ej_rollout_noalloc(E: int, N: int, R: int, params: EjParams, seed: int, T: int, actions: int | None, gov_actions: int | None,
                       obs_ring: int | None, rew_ring: int | None, done_ring: int | None, cuda_stream: int | None):
    _check(None, lib().ej_rollout_noalloc(E, N, R, C.byref(params), C.c_uint64(seed), T, actions, gov_actions, obs_ring, rew_ring,
                                          done_ring, cuda_stream))


def ej_launch_count(h) -> int:
    return int(lib().ej_launch_count(h))


def _dp(t):
    return None if t is None else t.data_ptr()


class Env:
    """Owns one ej_env handle and the PyTorch tensors its calls read and write."""

    def __init__(self, E: int, N: int, R: int, params: dict, device: str = "cuda:0"):
        import torch

        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.params = dict(params)
        self.h = ej_create(E, N, R, make_params(params))
        self.info = ej_layout(self.h)
        for k, _ in EjLayoutInfo._fields_:
            setattr(self, k, getattr(self.info, k))
        ej_set_stream(self.h, torch.cuda.current_stream(self.device).cuda_stream)

    def close(self):
        if getattr(self, "h", None):
            ej_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def use_current_stream(self):
        ej_set_stream(self.h, self.torch.cuda.current_stream(self.device).cuda_stream)

    def reset(self, seed: int):
        ej_reset(self.h, seed)

    # -- tensor allocation helpers --
    def new_obs(self, depth=None):
        shape = (self.obs_floats,) if depth is None else (depth, self.obs_floats)
        return self.torch.zeros(shape, dtype=self.torch.float32, device=self.device)

    def new_rew(self, depth=None):
        shape = (self.E, self.N + 1) if depth is None else (depth, self.E, self.N + 1)
        return self.torch.zeros(shape, dtype=self.torch.float32, device=self.device)

    def new_done(self, depth=None):
        shape = (self.E,) if depth is None else (depth, self.E)
        return self.torch.zeros(shape, dtype=self.torch.uint8, device=self.device)

    def split_obs(self, obs):
        """Views (pop [.., E, N, D_pop], gov [.., E, D_gov]) of an obs buffer or ring."""
        lead = obs.shape[:-1]
        pop = obs[..., : self.E * self.N * self.D_pop].reshape(*lead, self.E, self.N, self.D_pop)
        gov = obs[..., self.gov_obs_offset:].reshape(*lead, self.E, self.D_gov_pad)[..., : self.D_gov]
        return pop, gov

    def observe(self, obs=None):
        obs = self.new_obs() if obs is None else obs
        ej_observe(self.h, obs.data_ptr())
        return obs

    def set_action_masking(self, on=True):
        ej_set_action_masking(self.h, on)

    def action_mask(self, mask=None):
        """f1: [E, N, A] uint8 availability mask of the current state."""
        t = self.torch
        if mask is None:
            mask = t.empty((self.E, self.N, self.A), dtype=t.uint8, device=self.device)
        assert mask.dtype == t.uint8 and mask.is_cuda and mask.is_contiguous() and mask.numel() == self.E * self.N * self.A
        ej_action_mask(self.h, mask.data_ptr())
        return mask

    def step(self, actions, gov_actions, obs=None, rew=None, done=None, want_obs=True):
        t = self.torch
        assert actions.dtype == t.int32 and actions.is_cuda and actions.is_contiguous() and actions.numel() == self.E * self.N
        assert gov_actions.dtype == t.int32 and gov_actions.is_cuda and gov_actions.is_contiguous() and gov_actions.numel() == self.E * self.B
        if obs is None and want_obs:
            obs = self.new_obs()
        rew = self.new_rew() if rew is None else rew
        done = self.new_done() if done is None else done
        ej_step(self.h, actions.data_ptr(), gov_actions.data_ptr(), _dp(obs), _dp(rew), _dp(done))
        return obs, rew, done

    def _host_in(self, a, n):
        """Host input as contiguous int32 (numpy's default integer is 64-bit: convert, never reinterpret)."""
        a = np.ascontiguousarray(a, np.int32)
        assert a.size == n, "expected %d int32 values, got %d" % (n, a.size)
        return a

    @staticmethod
    def _host_out(a, dtype, n, what):
        """Host output buffer the library writes through a raw pointer: dtype, size and contiguity are checked."""
        if a is None:
            return None
        assert isinstance(a, np.ndarray) and a.dtype == dtype and a.flags["C_CONTIGUOUS"] and a.flags["WRITEABLE"] and a.size >= n, \
            "%s must be a writable C-contiguous %s array of at least %d elements" % (what, np.dtype(dtype).name, n)
        return a.ctypes.data

    def step_host(self, actions: np.ndarray, gov_actions: np.ndarray, obs: np.ndarray | None, rew: np.ndarray | None,
                  done: np.ndarray | None):
        a, g = self._host_in(actions, self.E * self.N), self._host_in(gov_actions, self.E * self.B)
        ej_step_host(self.h, a.ctypes.data, g.ctypes.data, self._host_out(obs, np.float32, self.obs_floats, "obs"),
                     self._host_out(rew, np.float32, self.rew_floats, "rew"), self._host_out(done, np.uint8, self.E, "done"))

    def step_host_factored(self, actions: np.ndarray, gov_actions: np.ndarray, priv: np.ndarray, shared: np.ndarray,
                           gov_obs: np.ndarray | None = None, rew: np.ndarray | None = None, done: np.ndarray | None = None):
        a, g = self._host_in(actions, self.E * self.N), self._host_in(gov_actions, self.E * self.B)
        ej_step_host_factored(self.h, a.ctypes.data, g.ctypes.data,
                              self._host_out(priv, np.float32, self.E * self.N * self.D_priv, "priv"),
                              self._host_out(shared, np.float32, self.E * self.D_shared_pad, "shared"),
                              self._host_out(gov_obs, np.float32, self.E * self.D_gov_pad, "gov_obs"),
                              self._host_out(rew, np.float32, self.rew_floats, "rew"), self._host_out(done, np.uint8, self.E, "done"))

    def set_policy(self, pop_net: dict | None, gov_net: dict | None):
        if pop_net is None and gov_net is None:
            ej_set_policy(self.h, None, None)
        else:
            ej_set_policy(self.h, make_mlp(pop_net), make_mlp(gov_net))

    def policy_act(self, obs, actions=None, gov_actions=None, pop_logits=None, gov_logits=None):
        t = self.torch
        actions = t.zeros((self.E, self.N), dtype=t.int32, device=self.device) if actions is None else actions
        gov_actions = t.zeros((self.E, self.B), dtype=t.int32, device=self.device) if gov_actions is None else gov_actions
        ej_policy_act(self.h, obs.data_ptr(), actions.data_ptr(), gov_actions.data_ptr(), _dp(pop_logits), _dp(gov_logits))
        return actions, gov_actions

    def rollout(self, T, ring_depth=1, actions_in=None, gov_actions_in=None, obs_ring=None, rew_ring=None,
                done_ring=None, actions_ring=None, gov_actions_ring=None, pop_logits_ring=None, gov_logits_ring=None,
                obs_priv_ring=None, obs_shared_ring=None, obs_gov_ring=None, auto_reset=False):
        io = EjRolloutIO()
        io.struct_size = C.sizeof(EjRolloutIO)
        io.ring_depth = ring_depth
        io.actions_in, io.gov_actions_in = _dp(actions_in), _dp(gov_actions_in)
        io.obs_ring, io.rew_ring, io.done_ring = _dp(obs_ring), _dp(rew_ring), _dp(done_ring)
        io.actions_ring, io.gov_actions_ring = _dp(actions_ring), _dp(gov_actions_ring)
        io.pop_logits_ring, io.gov_logits_ring = _dp(pop_logits_ring), _dp(gov_logits_ring)
        io.obs_priv_ring, io.obs_shared_ring, io.obs_gov_ring = _dp(obs_priv_ring), _dp(obs_shared_ring), _dp(obs_gov_ring)
        io.auto_reset = 1 if auto_reset else 0
        ej_rollout(self.h, T, io)

    # f2, factored observations: the three rings of one step (widths from ej_layout)
    def new_factored_obs(self, depth=1):
        t = self.torch
        z = lambda *shape: t.zeros(shape, dtype=t.float32, device=self.device)
        return z(depth, self.E, self.N, self.D_priv), z(depth, self.E, self.D_shared_pad), z(depth, self.E, self.D_gov_pad)

    def set_action_cdf(self, cdf: np.ndarray):
        cdf = np.ascontiguousarray(cdf, np.uint32)
        ej_set_action_cdf(self.h, cdf.ctypes.data, int(cdf.shape[0]))

    def get_state(self, env_begin=0, env_count=None) -> np.ndarray:
        n = self.E - env_begin if env_count is None else env_count
        w = np.zeros((n, self.state_words), np.int32)
        ej_get_state(self.h, env_begin, n, w.ctypes.data, w.size)
        return w

    def set_state(self, words: np.ndarray, env_begin=0):
        words = np.ascontiguousarray(words, np.int32)
        ej_set_state(self.h, env_begin, words.shape[0], words.ctypes.data, words.size)

    def launch_count(self) -> int:
        return ej_launch_count(self.h)
