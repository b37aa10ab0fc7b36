"""Helpers of the GPU parity tests: run the CUDA path (through the C ABI) and the CPU oracle on
the same seeded inputs and compare them element by element.

Tolerances (BASELINE.json north_star): integer state, books, counters and
the binary32 agent state (coin, labor, income, skills, rates) bit-exact; rewards and the
government mean / std within 1e-6 + 1e-5 * |oracle|; medians and every population
observation entry exact.
"""
import numpy as np

import oracle
from paper_2410_22165_b200 import binding

RTOL, ATOL = 1e-5, 1e-6


def close(a, b, what):
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
    bad = np.abs(a - b) > ATOL + RTOL * np.abs(b)
    assert not bad.any(), "%s: %d of %d outside tolerance, worst |d|=%g at %s (gpu %r, oracle %r)" % (
        what, bad.sum(), bad.size, np.abs(a - b).max(), np.argwhere(bad)[0], a[bad][0], b[bad][0])


def exact(a, b, what):
    a = np.asarray(a)
    b = np.asarray(b)
    assert a.shape == b.shape, "%s: shape %s vs %s" % (what, a.shape, b.shape)
    if a.dtype.kind == "f":
        same = a.view(np.uint32) == b.view(np.uint32)
    else:
        same = a == b
    assert same.all(), "%s: %d of %d differ, first at %s (gpu %r, oracle %r)" % (
        what, (~same).sum(), same.size, np.argwhere(~same)[0], a[~same][0], b[~same][0])


def compare_state(gw, ow, what="state"):
    """Canonical dumps [n][W]: everything bit-exact except u_g_prev (binary64, words 11-12)."""
    gw = np.asarray(gw)
    ow = np.asarray(ow)
    exact(gw[:, :11], ow[:, :11], what + " header/counters")
    exact(gw[:, 13:], ow[:, 13:], what + " body")
    close(gw[:, 11:13].copy().view(np.float64), ow[:, 11:13].copy().view(np.float64), what + " u_g_prev")


def compare_outputs(genv, g_obs_pop, g_obs_gov, g_rew, g_done, o_obs_pop, o_obs_gov, o_rew, o_done, what=""):
    """Observation / reward / done parity of one step for a set of envs."""
    R, B = genv.R, genv.B
    exact(g_done, o_done, what + " done")
    if o_obs_pop is not None:
        exact(g_obs_pop, o_obs_pop, what + " population observations")
        gg = g_obs_gov.reshape(-1, genv.D_gov)
        og = o_obs_gov.reshape(-1, genv.D_gov)
        nm = 3 + R
        stats_g = gg[:, : 3 * nm].reshape(-1, nm, 3)
        stats_o = og[:, : 3 * nm].reshape(-1, nm, 3)
        close(stats_g[:, :, 0], stats_o[:, :, 0], what + " gov mean")
        close(stats_g[:, :, 1], stats_o[:, :, 1], what + " gov std")
        exact(stats_g[:, :, 2], stats_o[:, :, 2], what + " gov median")
        exact(gg[:, 3 * nm:], og[:, 3 * nm:], what + " gov rates/timers")
    close(g_rew, o_rew, what + " rewards")


class Pair:
    """The CUDA env and the oracle on the same (E, N, R, params, seed)."""

    def __init__(self, E, N, R, params, seed, env_ids=None):
        import torch

        self.torch = torch
        self.g = binding.Env(E, N, R, params)
        self.g.reset(seed)
        self.seed = seed
        # oracle envs: all of them, or a subset of global env ids (each a 1-env oracle based at that id)
        self.env_ids = list(range(E)) if env_ids is None else list(env_ids)
        if env_ids is None:
            self.o = [oracle.OracleEnv(E, N, R, params)]
            self.o[0].reset(seed)
        else:
            base = int(params["env_id_base"])
            self.o = []
            for g in self.env_ids:
                o = oracle.OracleEnv(1, N, R, dict(params, env_id_base=base + g))
                o.reset(seed)
                self.o.append(o)
        self.full = env_ids is None

    def o_state(self):
        if self.full:
            return self.o[0].get_state()
        return np.concatenate([o.get_state() for o in self.o])

    def g_state(self):
        if self.full:
            return self.g.get_state()
        return np.concatenate([self.g.get_state(e, 1) for e in self.env_ids])

    def o_step(self, acts, gov, want_obs=True):
        if self.full:
            return self.o[0].step(acts, gov, want_obs=want_obs)
        outs = [o.step(acts[e:e + 1], gov[e:e + 1], want_obs=want_obs) for o, e in zip(self.o, self.env_ids)]
        cat = lambda k: None if outs[0][k] is None else np.concatenate([x[k] for x in outs])
        return cat(0), cat(1), cat(2), cat(3)

    def o_draw(self, cdf):
        if self.full:
            return self.o[0].draw_actions(cdf)
        outs = [o.draw_actions(cdf) for o in self.o]
        return np.concatenate([x[0] for x in outs]), np.concatenate([x[1] for x in outs])

    def step_and_compare(self, acts, gov, what="", check_state=True, want_obs=True):
        t = self.torch
        g_obs, g_rew, g_done = self.g.step(t.from_numpy(np.ascontiguousarray(acts)).cuda(),
                                           t.from_numpy(np.ascontiguousarray(gov)).cuda(), want_obs=want_obs)
        o_pop, o_gov, o_rew, o_done = self.o_step(acts, gov, want_obs=want_obs)
        ids = self.env_ids
        if want_obs:
            pop, gv = self.g.split_obs(g_obs)
            pop, gv = pop.cpu().numpy()[ids], gv.cpu().numpy()[ids]
        else:
            pop = gv = None
        compare_outputs(self.g, pop, gv, g_rew.cpu().numpy()[ids], g_done.cpu().numpy()[ids], o_pop, o_gov, o_rew,
                        o_done, what)
        if check_state:
            compare_state(self.g_state(), self.o_state(), what + " state")
