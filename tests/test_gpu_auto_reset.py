"""f4 slice (G44): ej_rollout with auto_reset against the oracle's orc_step_auto.  An env
whose episode ends starts the next one inside the same step; every draw of the new episode is keyed by its index; the
step that ends an episode returns its own rewards and done and the fresh state's observation."""
import numpy as np
import pytest

import oracle
from paper_2410_22165_b200 import binding, inputs
from parity import Pair, compare_outputs, compare_state, exact

pytestmark = pytest.mark.gpu


def _auto(name, E, steps, supplied=False, ring=None, factored=False, **over):
    import torch

    cfg = inputs.configs()[name]
    params = dict(cfg["params"], **over)
    cfg = dict(cfg, params=params)
    N, T = cfg["N"], params["episode_length"]
    pair = Pair(E, N, cfg["R"], params, cfg["seed"])
    g, o = pair.g, pair.o[0]
    cdf = inputs.action_cdf(cfg)
    g.set_action_cdf(cdf)
    depth = steps if ring is None else ring
    obs_ring, rew_ring, done_ring = g.new_obs(depth), g.new_rew(depth), g.new_done(depth)
    act_ring = torch.zeros((depth, E, N), dtype=torch.int32, device="cuda")
    gov_ring = torch.zeros((depth, E, g.B), dtype=torch.int32, device="cuda")
    kw = {}
    if supplied:
        acts, gov = inputs.action_stream(cfg, steps, seed=3, E=E)
        kw = dict(actions_in=torch.from_numpy(acts).cuda(), gov_actions_in=torch.from_numpy(gov).cuda())
    g.rollout(steps, ring_depth=depth, obs_ring=obs_ring, rew_ring=rew_ring, done_ring=done_ring, actions_ring=act_ring,
              gov_actions_ring=gov_ring, auto_reset=True, **kw)
    torch.cuda.synchronize()
    pop, gv = g.split_obs(obs_ring)
    pop, gv, rew, done = pop.cpu().numpy(), gv.cpu().numpy(), rew_ring.cpu().numpy(), done_ring.cpu().numpy()
    a_out, g_out = act_ring.cpu().numpy(), gov_ring.cpu().numpy()
    n_done = 0
    for t in range(steps):
        if supplied:
            o_a, o_g = acts[t], gov[t]
        else:
            o_a, o_g = o.draw_actions(cdf)
        o_pop, o_gov, o_rew, o_done = o.step(o_a, o_g, auto_reset=True)
        n_done += int(o_done.sum())
        if t >= steps - depth:
            slot = t % depth
            exact(a_out[slot], o_a, "%s t=%d actions" % (name, t))
            exact(g_out[slot], o_g, "%s t=%d government levels" % (name, t))
            compare_outputs(g, pop[slot], gv[slot], rew[slot], done[slot], o_pop, o_gov, o_rew, o_done, "%s auto-reset t=%d" % (name, t))
    compare_state(pair.g_state(), pair.o_state(), name + " state after the auto-resetting rollout")
    assert n_done == E * (steps // T)
    ep = [oracle.parse_state(w)["episode"] for w in pair.g_state()]
    assert ep == [steps // T] * E
    return pair


def test_auto_reset_tiny_two_episodes_and_a_bit():
    _auto("tiny_dense", 8, 2 * 50 + 7)
    _auto("config1_tiny", 1, 3 * 50)


def test_auto_reset_paper_shape_short_episodes():
    # the shape-specialised kernel (16-bit order pool), episodes of 70 steps with a tax collection at the boundary
    _auto("config2_paper", 6, 3 * 70 + 11, episode_length=70, tax_period=35)
    _auto("config2_paper", 4, 2 * 45 + 5, supplied=True, ring=6, episode_length=45, tax_period=15)


def test_auto_reset_resource_and_population_scaling_shapes():
    _auto("config3_resources", 3, 2 * 40 + 3, episode_length=40, tax_period=20)
    _auto("section5_r12", 2, 2 * 30 + 2, episode_length=30)                  # generic kernel, growing skills
    _auto("config4_population", 2, 2 * 35 + 4, episode_length=35, tax_period=35)  # 1024-thread CTA: bucketed statistics, row buffers


def test_auto_reset_in_split_calls_and_after_a_finished_episode():
    import torch

    cfg = inputs.configs()["tiny_dense"]
    T = cfg["T"]
    a = binding.Env(5, cfg["N"], cfg["R"], cfg["params"])
    b = binding.Env(5, cfg["N"], cfg["R"], cfg["params"])
    a.reset(9)
    b.reset(9)
    a.rollout(2 * T + 20, auto_reset=True)
    b.rollout(T - 3, auto_reset=True)
    b.rollout(3)                       # the episode ends in a call without auto-reset: the envs stay done (G28) ...
    b.rollout(2)                       # ... and stepping them changes nothing
    assert (b.get_state()[:, 0] == T).all()
    b.rollout(T + 20, auto_reset=True)   # the next auto-resetting call starts episode 1 with its first step
    torch.cuda.synchronize()
    exact(a.get_state(), b.get_state(), "auto-reset in one call / in split calls")


def test_auto_reset_policy_rollout_teacher_forced():
    """Policy mode: the policy acts on the fresh state's observation after an episode ends; sampling is keyed by the episode."""
    import torch
    from oracle import policy as OP

    cfg = inputs.configs()["config5_policy"]
    N, R, E, T = cfg["N"], cfg["R"], 3, 24
    params = dict(cfg["params"], episode_length=T, tax_period=12)
    pair = Pair(E, N, R, params, 4)
    g, o = pair.g, pair.o[0]
    pop, gov = inputs.policy_weights(cfg, seed=2, std=0.3, bias_std=0.1)
    g.set_policy(pop, gov)
    steps = 2 * T + 5
    obs_ring, rew_ring, done_ring = g.new_obs(steps), g.new_rew(steps), g.new_done(steps)
    act_ring = torch.zeros((steps, E, N), dtype=torch.int32, device="cuda")
    gov_ring = torch.zeros((steps, E, g.B), dtype=torch.int32, device="cuda")
    pl_ring = torch.zeros((steps, E * N, g.A), dtype=torch.float32, device="cuda")
    g.rollout(steps, ring_depth=steps, obs_ring=obs_ring, rew_ring=rew_ring, done_ring=done_ring, actions_ring=act_ring,
              gov_actions_ring=gov_ring, pop_logits_ring=pl_ring, auto_reset=True)
    torch.cuda.synchronize()
    popo, gvo = g.split_obs(obs_ring)
    popo, gvo, rew, done = popo.cpu().numpy(), gvo.cpu().numpy(), rew_ring.cpu().numpy(), done_ring.cpu().numpy()
    a_out, g_out = act_ring.cpu().numpy(), gov_ring.cpu().numpy()
    pl = pl_ring.cpu().numpy().reshape(steps, E, N, -1)
    o_pop, o_gov = o.observe()
    for t in range(steps):
        ol = OP.mlp_logits(pop, o_pop.reshape(E * N, -1)).reshape(E, N, -1)
        assert np.abs(pl[t] - ol).max() <= 2e-2 * np.abs(ol).max() + 1e-3, "t=%d logits" % t
        ep, tt = divmod(t, T)
        for e in range(E):      # the draw is keyed by (t within the episode, stream | episode << 8)
            u = OP.philox_u(4, e, 7, tt, 0 | (ep << 8), 0)
            assert OP.sample_consistent(ol[e, 7], u, int(a_out[t, e, 7]), 1e-3), "t=%d env %d" % (t, e)
        o_pop, o_gov, o_rew, o_done = o.step(a_out[t], g_out[t], auto_reset=True)
        compare_outputs(g, popo[t], gvo[t], rew[t], done[t], o_pop, o_gov, o_rew, o_done, "policy auto-reset t=%d" % t)
    compare_state(pair.g_state(), pair.o_state(), "policy auto-reset final state")
    assert done.sum() == 2 * E
