"""f2 parity: factored observations of ej_rollout against the oracle's observation, column for
column: priv[e][i][k] = obs row (e, i) column k for k < 3R + 4; shared[e][k] = column 3R + 4 + k of
every row of env e (market statistics, tax rates and timers are env-wide)."""
import numpy as np
import pytest

from paper_2410_22165_b200 import binding, inputs

pytestmark = pytest.mark.gpu


def _run(name, E, T, params_over=None, seed=4, N=None):
    import torch
    from parity import Pair, close, compare_state, exact

    cfg = inputs.configs()[name]
    if N is not None:
        cfg = dict(cfg, N=N)
    params = dict(cfg["params"], **(params_over or {}))
    pair = Pair(E, cfg["N"], cfg["R"], params, seed)
    g = pair.g
    acts, gov = inputs.action_stream(dict(cfg, params=params), T, seed=seed, E=E)
    priv, shared, govr = g.new_factored_obs(T)
    rew = g.new_rew(T)
    g.rollout(T, ring_depth=T, actions_in=torch.from_numpy(acts).cuda(), gov_actions_in=torch.from_numpy(gov).cuda(),
              rew_ring=rew, obs_priv_ring=priv, obs_shared_ring=shared, obs_gov_ring=govr)
    torch.cuda.synchronize()
    priv, shared, govr, rew = priv.cpu().numpy(), shared.cpu().numpy(), govr.cpu().numpy(), rew.cpu().numpy()
    dp, ds = g.D_priv, g.D_shared
    assert dp + ds == g.D_pop
    for t in range(T):
        o_pop, o_gov, o_rew, _ = pair.o[0].step(acts[t], gov[t])
        exact(priv[t], o_pop[:, :, :dp], "%s t=%d private block" % (name, t))
        exact(shared[t][:, :ds], o_pop[:, 0, dp:], "%s t=%d env-wide block" % (name, t))
        close(govr[t][:, : g.D_gov], o_gov, "%s t=%d government rows" % (name, t))
        close(rew[t], o_rew, "%s t=%d rewards" % (name, t))
    compare_state(pair.g_state(), pair.o_state(), name + " state after the factored rollout")


def test_factored_generic_kernel_small_population():
    _run("config2_paper", 4, 60, dict(tax_period=20), N=32)   # 32-thread CTAs, generic variant


def test_factored_paper_shape_specialised_kernel():
    _run("config2_paper", 5, 130, dict(tax_period=25))


def test_factored_six_resources():
    _run("config3_resources", 3, 60, dict(tax_period=20))


def test_factored_with_growing_skills():
    # f3 under f2: the skill columns of the private block change at any step
    _run("config2_paper", 4, 80, dict(tax_period=25, skill_growth_rate=0.005, skill_max=5.0))
    _run("section5_r4", 3, 60)


def test_step_host_factored_against_the_oracle():
    # ej_step_host_factored: host buffers in and out, one step per call; every column against the oracle's dense rows
    from parity import Pair, close, compare_state, exact

    for name, E, over in (("config2_paper", 4, dict(tax_period=10)), ("section5_r4", 3, {})):
        cfg = inputs.configs()[name]
        params = dict(cfg["params"], **over)
        pair = Pair(E, cfg["N"], cfg["R"], params, 8)
        g = pair.g
        acts, gov = inputs.action_stream(dict(cfg, params=params), 35, seed=8, E=E)
        priv = np.zeros((E, cfg["N"], g.D_priv), np.float32)
        shared = np.zeros((E, g.D_shared_pad), np.float32)
        govr = np.zeros((E, g.D_gov_pad), np.float32)
        rew = np.zeros((E, cfg["N"] + 1), np.float32)
        done = np.zeros(E, np.uint8)
        for t in range(35):
            if t % 2:
                g.step_host_factored(acts[t], gov[t], priv, shared, govr, rew, done)
            else:   # optional outputs left out
                g.step_host_factored(acts[t], gov[t], priv, shared)
            o_pop, o_gov, o_rew, o_done = pair.o[0].step(acts[t], gov[t])
            exact(priv, o_pop[:, :, : g.D_priv], "%s t=%d private block" % (name, t))
            exact(shared[:, : g.D_shared], o_pop[:, 0, g.D_priv:], "%s t=%d env-wide block" % (name, t))
            if t % 2:
                close(govr[:, : g.D_gov], o_gov, "%s t=%d government rows" % (name, t))
                close(rew, o_rew, "%s t=%d rewards" % (name, t))
                exact(done, o_done.astype(np.uint8), "%s t=%d done" % (name, t))
        compare_state(pair.g_state(), pair.o_state(), name + " state after host factored steps")
        with pytest.raises(binding.EjError):
            binding.ej_step_host_factored(g.h, acts[0].ctypes.data, gov[0].ctypes.data, priv.ctypes.data, None, None, None, None)


def test_factored_errors():
    import torch

    cfg = inputs.configs()["tiny_dense"]
    env = binding.Env(2, cfg["N"], cfg["R"], cfg["params"])
    env.reset(1)
    priv, shared, govr = env.new_factored_obs(1)
    with pytest.raises(binding.EjError):
        env.rollout(1, obs_priv_ring=priv)                                         # the env-wide block is missing
    with pytest.raises(binding.EjError):
        env.rollout(1, obs_ring=env.new_obs(1), obs_priv_ring=priv, obs_shared_ring=shared)  # both layouts at once
    big = inputs.configs()["config4_population"]
    env4 = binding.Env(1, big["N"], big["R"], big["params"])
    env4.reset(1)
    p4, s4, g4 = env4.new_factored_obs(1)
    with pytest.raises(binding.EjError):
        env4.rollout(1, obs_priv_ring=p4, obs_shared_ring=s4)                       # N = 1000: tile not staged
    torch.cuda.synchronize()
