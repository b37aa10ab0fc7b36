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


def check_dump_invariants(w, cfg, steps):
    """What the rules fix at any size, checked vectorised on the canonical dump `w`
    (int32 [E][state_words]) of envs that ran `steps` steps: escrow = sum of the agent's live orders, live-order
    counts and cap, ages below the expiry, books in priority order and uncrossed,
    prices on the grid, nothing negative, clock and counters consistent."""
    E, N, R, p = w.shape[0], cfg["N"], cfg["R"], cfg["params"]
    B, P, M = len(p["thresholds"]) + 1, len(p["prices"]), p["max_active_orders"]
    cap = int(w[0, 5])
    assert (w[:, 0] == steps).all() and (w[:, 1] == N).all() and (w[:, 2] == R).all() and (w[:, 3] == B).all() and (w[:, 4] == P).all()
    q = 13 + B + R
    rec = 6 + 3 * R
    ag = w[:, q:q + N * rec].reshape(E, N, rec)
    q += N * rec
    f32 = lambda a: np.ascontiguousarray(a, np.int32).view(np.float32)
    coin, labor = f32(ag[:, :, 0]), f32(ag[:, :, 3])
    esc_coin, n_live = ag[:, :, 1], ag[:, :, 5]
    inv, esc_res = ag[:, :, 6:6 + R], ag[:, :, 6 + R:6 + 2 * R]
    assert (coin >= 0).all() and np.isfinite(coin).all() and (labor >= 0).all()
    assert (inv >= 0).all() and (esc_res >= 0).all() and (esc_coin >= 0).all()
    live = np.zeros((E, N), np.int64)
    want_coin = np.zeros((E, N), np.int64)
    want_res = np.zeros((E, N, R), np.int64)
    env_idx = np.repeat(np.arange(E), cap).reshape(E, cap)
    best = {}
    n_orders = 0
    for b in range(2 * R):
        n = w[:, q]
        book = w[:, q + 1:q + 1 + 3 * cap].reshape(E, cap, 3)
        q += 1 + 3 * cap
        assert (n >= 0).all() and (n <= cap).all()
        valid = np.arange(cap)[None, :] < n[:, None]
        price, owner, placed = book[:, :, 0][valid], book[:, :, 1][valid], book[:, :, 2][valid]
        e_of = env_idx[valid]
        n_orders += int(valid.sum())
        assert np.isin(price, p["prices"]).all() and (owner >= 0).all() and (owner < N).all()
        age = (steps - 1) - placed
        assert (age >= 0).all() and (age < p["order_expiry"]).all()
        np.add.at(live, (e_of, owner), 1)
        if b % 2 == 0:
            np.add.at(want_coin, (e_of, owner), price.astype(np.int64))
        else:
            np.add.at(want_res, (e_of, owner, b // 2), 1)
        # priority order: bids by falling price, asks by rising price; among equal prices the older order first
        pr = np.where(valid, book[:, :, 0], np.int32(-1 if b % 2 == 0 else 1 << 20))
        d = np.diff(pr, axis=1)
        assert (d <= 0).all() if b % 2 == 0 else (d >= 0).all()
        both = valid[:, 1:] & valid[:, :-1] & (d == 0)
        assert (np.diff(book[:, :, 2], axis=1)[both] >= 0).all()
        best[b] = np.where(n > 0, book[:, 0, 0], -1)
    assert q + 1 == w.shape[1] and (w[:, q] >= 0).all()             # last word: episode index (f4)
    assert (want_coin == esc_coin).all() and (want_res == esc_res).all()            # escrow = sum of live orders
    assert (live == n_live).all() and live.max() <= M
    for r in range(R):                                                               # uncrossed after matching
        bb, ab = best[2 * r], best[2 * r + 1]
        both = (bb >= 0) & (ab >= 0)
        assert (bb[both] < ab[both]).all()
    return n_orders


class OracleShards:
    """The oracle on runs of consecutive global env ids, advanced by host threads (economies are independent and
    keyed by their global id; ctypes releases the GIL while the C oracle steps).  Used by the full-size parity tests:
    the oracle itself is unchanged, only many copies of it run side by side."""

    def __init__(self, N, R, params, seed, runs, threads=None, per_shard=None):
        import os
        from concurrent.futures import ThreadPoolExecutor

        self.N, self.R = N, R
        self.runs = [(int(lo), int(n)) for lo, n in runs]
        total = sum(n for _, n in self.runs)
        self.threads = threads or max(1, min(os.cpu_count() or 1, 32))
        per = per_shard or max(1, -(-total // (4 * self.threads)))
        self.shards = []   # (first local index in the concatenated order, oracle env)
        k = 0
        base = int(params["env_id_base"])
        for lo, n in self.runs:
            for s in range(lo, lo + n, per):
                cnt = min(per, lo + n - s)
                o = oracle.OracleEnv(cnt, N, R, dict(params, env_id_base=base + s))
                o.reset(seed)
                self.shards.append((k, o))
                k += cnt
        self.n = k
        self.ids = np.concatenate([np.arange(lo, lo + n) for lo, n in self.runs])
        self.pool = ThreadPoolExecutor(self.threads)

    def _map(self, fn):
        return list(self.pool.map(fn, self.shards))

    def state(self):
        return np.concatenate(self._map(lambda s: s[1].get_state()))

    def observe(self):
        outs = self._map(lambda s: s[1].observe())
        return np.concatenate([x[0] for x in outs]), np.concatenate([x[1] for x in outs])

    def advance(self, steps, cdf=None, actions=None, gov_actions=None, keep=()):
        """Step every env `steps` times with actions drawn from `cdf` (rollout-mode generator) or supplied as
        [steps][n][N] / [steps][n][B] in the concatenated env order.  Returns {s: (acts, gov, pop, govobs, rew, done)}
        for the step indices s in `keep` (observations are built only there)."""
        keep = set(keep)

        def work(sh):
            k, o = sh
            out = {}
            for s in range(steps):
                if actions is None:
                    a, g = o.draw_actions(cdf)
                else:
                    a, g = actions[s][k:k + o.E], gov_actions[s][k:k + o.E]
                pop, gv, rew, done = o.step(a, g, want_obs=s in keep)
                if s in keep:
                    out[s] = (a, g, pop, gv, rew, done)
            return out

        parts = self._map(work)
        return {s: tuple(np.concatenate([p[s][j] for p in parts]) for j in range(6)) for s in keep}
