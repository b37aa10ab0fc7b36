"""Full-size GPU parity (SURVEY.md 8(d) "Parity runs on all envs for configs 1 and 2; on envs {0..127} U
{E-128..E-1} for configs 3 and 4; config 5 teacher-forced on envs 0..127"): every config in the launch
configuration bench.py times (ej_rollout, persistent kernel, generated actions, output rings), run to the end of
the episode, against the CPU oracle sharded over the host cores.  Canonical dumps are compared every 100 steps and
at t = T; actions, observations, rewards and done on the last steps of every 100-step chunk."""
import numpy as np
import pytest

from paper_2410_22165_b200 import binding, inputs
from parity import OracleShards, compare_outputs, compare_state, exact

pytestmark = pytest.mark.gpu


def _g_state(g, runs):
    return np.concatenate([g.get_state(lo, n) for lo, n in runs])


def _full_size(name, runs, T=None, chunk=100, keep=2):
    import torch

    cfg = inputs.configs()[name]
    E, N, R = cfg["E"], cfg["N"], cfg["R"]
    T = cfg["T"] if T is None else T
    g = binding.Env(E, N, R, cfg["params"])
    g.reset(cfg["seed"])
    cdf = inputs.action_cdf(cfg)
    g.set_action_cdf(cdf)
    o = OracleShards(N, R, cfg["params"], cfg["seed"], runs)
    ids = torch.from_numpy(o.ids).cuda()
    compare_state(_g_state(g, runs), o.state(), name + " reset")
    obs_ring, rew_ring, done_ring = g.new_obs(keep), g.new_rew(keep), g.new_done(keep)
    act_ring = torch.zeros((keep, E, N), dtype=torch.int32, device="cuda")
    gov_ring = torch.zeros((keep, E, g.B), dtype=torch.int32, device="cuda")
    t = 0
    while t < T:
        m = min(chunk, T - t)
        g.rollout(m, ring_depth=keep, obs_ring=obs_ring, rew_ring=rew_ring, done_ring=done_ring, actions_ring=act_ring,
                  gov_actions_ring=gov_ring)
        kept = [s for s in range(max(0, m - keep), m)]
        outs = o.advance(m, cdf=cdf, keep=kept)
        torch.cuda.synchronize()
        pop, gv = g.split_obs(obs_ring)
        for s in kept:
            slot = s % keep
            o_a, o_g, o_pop, o_gov, o_rew, o_done = outs[s]
            what = "%s t=%d" % (name, t + s)
            exact(act_ring[slot][ids].cpu().numpy(), o_a, what + " generated actions")
            exact(gov_ring[slot][ids].cpu().numpy(), o_g, what + " generated government levels")
            compare_outputs(g, pop[slot][ids].cpu().numpy(), gv[slot][ids].cpu().numpy(), rew_ring[slot][ids].cpu().numpy(),
                            done_ring[slot][ids].cpu().numpy(), o_pop, o_gov, o_rew, o_done, what)
        t += m
        compare_state(_g_state(g, runs), o.state(), "%s state at t=%d" % (name, t))
    w = _g_state(g, runs)
    assert (w[:, 0] == T).all()                                  # every env finished its episode ...
    assert (w[:, 6] > 0).all() or name == "config1_tiny"        # ... and traded (literal config 1 never does: G38)
    return g, o


def _ends(E, n=128):
    return [(0, n), (E - n, n)]


def test_config2_every_env_full_episode():
    _full_size("config2_paper", [(0, 1024)])


def test_headline_first_and_last_128_envs_full_episode():
    g, o = _full_size("headline", _ends(4096))
    # a finished env is a no-op (G28): 3 more steps change nothing and report done
    import torch
    before = _g_state(g, o.runs)
    done = g.new_done(1)
    g.rollout(3, ring_depth=1, done_ring=done)
    torch.cuda.synchronize()
    exact(_g_state(g, o.runs), before, "state after stepping finished envs")
    assert (done.cpu().numpy() == 1).all()


def test_config3_first_and_last_128_envs_full_episode():
    _full_size("config3_resources", _ends(4096))


def test_config4_every_env_full_episode():
    # N = 1000 with the book cap K = N (G15): all 256 envs, the path with the most code of its own
    _full_size("config4_population", [(0, 256)], chunk=125)


def test_section5_shapes_first_and_last_64_envs_half_episode():
    _full_size("section5_r4", _ends(4096, 64), T=500)
    _full_size("section5_r12", _ends(2048, 64), T=300)


def test_config1_tiny_literal():
    _full_size("config1_tiny", [(0, 1)], chunk=10)
