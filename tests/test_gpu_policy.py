"""GPU parity of a12 (policy MLP on the tensor cores + categorical sampling) against
oracle/policy.py, and the teacher-forced rollout protocol of DESIGN.md G33: the oracle env
consumes the actions the GPU sampled, every transition / observation / reward is compared as in
test_gpu_parity.py, the logits are recomputed in binary64 from the (bit-identical) observations,
and each sampled action must lie in its CDF interval widened by eps."""
import numpy as np
import pytest

import oracle
from oracle import policy as OP
from paper_2410_22165_b200 import binding, inputs
from parity import Pair, compare_outputs, compare_state, exact

pytestmark = pytest.mark.gpu

EPS_CDF = 1e-3        # G33: widening of the CDF interval
LOGIT_RTOL, LOGIT_ATOL = 2e-2, 1e-3   # G33: abs(d) <= 2e-2 * max abs(logit) + 1e-3


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")


def check_logits(g, o, what):
    g, o = np.asarray(g, np.float64), np.asarray(o, np.float64)
    tol = LOGIT_RTOL * np.abs(o).max() + LOGIT_ATOL
    err = np.abs(g - o).max()
    assert err <= tol, "%s: logits differ by %g (tolerance %g)" % (what, err, tol)
    return err / max(np.abs(o).max(), 1e-30)


def check_samples(seed, gids, N, t_of_env, pop_logits, gov_logits, acts, gov, B, L, what):
    """Every sampled action must be eps-consistent with the oracle's logits; returns the number of
    samples where the oracle's own draw differs (eps-ambiguous ones)."""
    ambiguous = total = 0
    for k, gid in enumerate(gids):
        t = int(t_of_env[k])
        for i in range(N):
            u = OP.philox_u(seed, gid, i, t, 0, 0)
            a = int(acts[k, i])
            assert OP.sample_consistent(pop_logits[k, i], u, a, EPS_CDF), "%s: env %d agent %d action %d not consistent with u=%g" % (what, gid, i, a, u)
            ambiguous += OP.sample(pop_logits[k, i], u) != a
            total += 1
        for b in range(B):
            u = OP.philox_u(seed, gid, N, t, 1 + b // 4, b % 4)
            a = int(gov[k, b])
            head = gov_logits[k, b * L:(b + 1) * L]
            assert OP.sample_consistent(head, u, a, EPS_CDF), "%s: env %d gov head %d level %d not consistent with u=%g" % (what, gid, b, a, u)
            ambiguous += OP.sample(head, u) != a
            total += 1
    return ambiguous, total


@pytest.mark.parametrize("std,bias_std,E", [(0.02, 0.0, 6), (0.3, 0.1, 3), (1.0, 0.5, 2)])
def test_policy_act_logits_and_samples(std, bias_std, E):
    import torch

    cfg = inputs.configs()["config5_policy"]
    N, R = cfg["N"], cfg["R"]
    params = dict(cfg["params"], env_id_base=11)
    pair = Pair(E, N, R, params, cfg["seed"])
    g = pair.g
    pop, gov = inputs.policy_weights(cfg, seed=1, std=std, bias_std=bias_std)
    g.set_policy(pop, gov)
    # a few random steps so that observations are not the reset state
    acts, govs = inputs.action_stream(cfg, 7, seed=2, E=E)
    for t in range(7):
        pair.step_and_compare(acts[t], govs[t], "warm t=%d" % t, check_state=False)
    obs = g.observe()
    pl = torch.zeros((E * N, g.A), dtype=torch.float32, device="cuda")
    gl = torch.zeros((E, g.B * g.L), dtype=torch.float32, device="cuda")
    a, gv = g.policy_act(obs, pop_logits=pl, gov_logits=gl)
    torch.cuda.synchronize()
    o_pop, o_gov = pair.o[0].observe()
    g_pop, g_gov = g.split_obs(obs)
    exact(g_pop.cpu().numpy(), o_pop, "observations fed to the policy")
    ol_pop = OP.mlp_logits(pop, o_pop.reshape(E * N, -1)).reshape(E, N, -1)
    ol_gov = OP.mlp_logits(gov, o_gov.reshape(E, -1))
    r1 = check_logits(pl.cpu().numpy().reshape(E, N, -1), ol_pop, "population logits")
    r2 = check_logits(gl.cpu().numpy(), ol_gov, "government logits")
    assert r1 < 5e-3 and r2 < 5e-3, "relative logit error %g / %g is far above bf16 re-rounding noise" % (r1, r2)
    amb, tot = check_samples(cfg["seed"], [11 + e for e in range(E)], N, [7] * E, ol_pop, ol_gov, a.cpu().numpy(),
                             gv.cpu().numpy(), g.B, g.L, "policy_act")
    assert amb <= max(2, 0.01 * tot), "%d of %d samples differ from the oracle's own draw" % (amb, tot)
    # the sampled actions are valid indices and not all equal
    an = a.cpu().numpy()
    assert an.min() >= 0 and an.max() < g.A and len(np.unique(an)) > 5


@pytest.mark.parametrize("over", [{}, dict(skill_growth_rate=0.005, skill_max=5.0)], ids=["fixed_skills", "growing_skills"])
def test_policy_rollout_teacher_forced(over):
    import torch

    cfg = inputs.configs()["config5_policy"]
    N, R, E, T = cfg["N"], cfg["R"], 5, 64
    params = dict(cfg["params"], tax_period=16, **over)   # f3: the policy observes skills that grow
    pair = Pair(E, N, R, params, cfg["seed"])
    g = pair.g
    pop, gov = inputs.policy_weights(cfg, seed=0, std=0.3, bias_std=0.1)  # non-uniform action distributions
    g.set_policy(pop, gov)
    obs0 = g.observe().clone()
    obs_ring, rew_ring, done_ring = g.new_obs(T), g.new_rew(T), g.new_done(T)
    act_ring = torch.zeros((T, E, N), dtype=torch.int32, device="cuda")
    gov_ring = torch.zeros((T, E, g.B), dtype=torch.int32, device="cuda")
    pl_ring = torch.zeros((T, E * N, g.A), dtype=torch.float32, device="cuda")
    gl_ring = torch.zeros((T, E, g.B * g.L), dtype=torch.float32, device="cuda")
    l0 = g.launch_count()
    g.rollout(T, ring_depth=T, obs_ring=obs_ring, rew_ring=rew_ring, done_ring=done_ring, actions_ring=act_ring,
              gov_actions_ring=gov_ring, pop_logits_ring=pl_ring, gov_logits_ring=gl_ring)
    torch.cuda.synchronize()
    assert g.launch_count() - l0 == 1 + 2 * T   # observe + (policy kernel, step kernel) per step
    pop_obs, gov_obs = g.split_obs(obs_ring)
    pop_obs, gov_obs = pop_obs.cpu().numpy(), gov_obs.cpu().numpy()
    rew, done = rew_ring.cpu().numpy(), done_ring.cpu().numpy()
    a_out, g_out = act_ring.cpu().numpy(), gov_ring.cpu().numpy()
    pl, gl = pl_ring.cpu().numpy().reshape(T, E, N, -1), gl_ring.cpu().numpy()
    o_pop, o_gov = pair.o[0].observe()
    p0, g0 = g.split_obs(obs0)
    exact(p0.cpu().numpy(), o_pop, "initial observation")
    amb = tot = 0
    worst = 0.0
    for t in range(T):
        # logits and samples from the observation of the state before step t (oracle's own, bit-identical)
        ol_pop = OP.mlp_logits(pop, o_pop.reshape(E * N, -1)).reshape(E, N, -1)
        ol_gov = OP.mlp_logits(gov, o_gov.reshape(E, -1))
        worst = max(worst, check_logits(pl[t], ol_pop, "t=%d population logits" % t), check_logits(gl[t], ol_gov, "t=%d government logits" % t))
        if t % 8 == 0 or t == T - 1:
            a_, t_ = check_samples(cfg["seed"], list(range(E)), N, [t] * E, ol_pop, ol_gov, a_out[t], g_out[t], g.B, g.L, "t=%d" % t)
            amb, tot = amb + a_, tot + t_
        # teacher forcing: the oracle env consumes the GPU's actions; transitions must match exactly
        o_pop, o_gov, o_rew, o_done = pair.o[0].step(a_out[t], g_out[t])
        compare_outputs(g, pop_obs[t], gov_obs[t], rew[t], done[t], o_pop, o_gov, o_rew, o_done, "policy rollout t=%d" % t)
    compare_state(pair.g_state(), pair.o_state(), "policy rollout final state")
    assert amb <= max(2, 0.01 * tot), "%d of %d samples differ from the oracle's own draw" % (amb, tot)
    assert worst < 5e-3
    # the policy really drove the economy: actions vary over agents and steps, and trades happened
    assert len(np.unique(a_out)) > 30
    s = oracle.parse_state(pair.g.get_state()[0])
    assert s["counters"][1] > 0


def test_policy_rollout_without_rings_matches_ringed_run():
    import torch

    cfg = inputs.configs()["config5_policy"]
    N, R, E, T = cfg["N"], cfg["R"], 3, 20
    pop, gov = inputs.policy_weights(cfg, seed=4, std=0.3)
    outs = []
    for ringed in (False, True):
        env = binding.Env(E, N, R, cfg["params"])
        env.reset(5)
        env.set_policy(pop, gov)
        if ringed:
            env.rollout(T, ring_depth=3, obs_ring=env.new_obs(3), rew_ring=env.new_rew(3), done_ring=env.new_done(3),
                        actions_ring=torch.zeros((3, E, N), dtype=torch.int32, device="cuda"),
                        gov_actions_ring=torch.zeros((3, E, env.B), dtype=torch.int32, device="cuda"))
        else:
            env.rollout(T)
        outs.append(env.get_state())
    exact(outs[0], outs[1], "policy rollout with / without output rings")


def test_policy_error_paths():
    cfg = inputs.configs()["config5_policy"]
    env = binding.Env(2, cfg["N"], cfg["R"], cfg["params"])
    env.reset(1)
    obs = env.observe()
    with pytest.raises(binding.EjError) as ei:
        env.policy_act(obs)
    assert ei.value.code == binding.EJ_ERR_STATE
    pop, gov = inputs.policy_weights(cfg, seed=0)
    bad = dict(pop, w1=pop["w1"][:, :-1])
    with pytest.raises(binding.EjError) as ei:
        env.set_policy(bad, gov)
    assert ei.value.code == binding.EJ_ERR_PARAM and "in_dim" in str(ei.value)
    bad = dict(gov, w3=gov["w3"][:-1], b3=gov["b3"][:-1])
    with pytest.raises(binding.EjError) as ei:
        env.set_policy(pop, bad)
    assert ei.value.code == binding.EJ_ERR_PARAM and "out_dim" in str(ei.value)
    env.set_policy(pop, gov)
    env.set_policy(None, None)
    with pytest.raises(binding.EjError):
        env.policy_act(obs)


def test_full_size_config5_envs_0_to_127_teacher_forced():
    """BASELINE.json configs[4] at full size (E=2048, N=100, R=3) in the launch configuration bench.py
    times (policy-driven ej_rollout with output rings), 200 steps; envs 0..127 are teacher-forced
    through the oracle sharded over the host cores: every transition, observation and reward of every step is
    compared, the logits are recomputed in binary64 every 8th step and the samples re-checked on a sample."""
    import torch
    from parity import OracleShards

    cfg = inputs.configs()["config5_policy"]
    N, R, E, T, chunk = cfg["N"], cfg["R"], cfg["E"], 200, 40
    n_ids = 128
    g = binding.Env(E, N, R, cfg["params"])
    g.reset(cfg["seed"])
    o = OracleShards(N, R, cfg["params"], cfg["seed"], [(0, n_ids)])
    pop, gov = inputs.policy_weights(cfg, seed=cfg["seed"])   # the weights bench.py installs
    g.set_policy(pop, gov)
    obs_ring, rew_ring, done_ring = g.new_obs(chunk), g.new_rew(chunk), g.new_done(chunk)
    act_ring = torch.zeros((chunk, E, N), dtype=torch.int32, device="cuda")
    gov_ring = torch.zeros((chunk, E, g.B), dtype=torch.int32, device="cuda")
    pl_ring = torch.zeros((chunk, E * N, g.A), dtype=torch.float32, device="cuda")
    gl_ring = torch.zeros((chunk, E, g.B * g.L), dtype=torch.float32, device="cuda")
    o_pop, o_gov = o.observe()
    amb = tot = 0
    worst = 0.0
    for c0 in range(0, T, chunk):
        g.rollout(chunk, ring_depth=chunk, obs_ring=obs_ring, rew_ring=rew_ring, done_ring=done_ring, actions_ring=act_ring,
                  gov_actions_ring=gov_ring, pop_logits_ring=pl_ring, gov_logits_ring=gl_ring)
        torch.cuda.synchronize()
        pop_obs, gov_obs = g.split_obs(obs_ring)
        pop_obs, gov_obs = pop_obs[:, :n_ids].cpu().numpy(), gov_obs[:, :n_ids].cpu().numpy()
        rew, done = rew_ring[:, :n_ids].cpu().numpy(), done_ring[:, :n_ids].cpu().numpy()
        a_out, g_out = act_ring[:, :n_ids].cpu().numpy(), gov_ring[:, :n_ids].cpu().numpy()
        # teacher forcing: the oracle envs consume the GPU's actions; every step's outputs are kept
        outs = o.advance(chunk, actions=a_out, gov_actions=g_out, keep=range(chunk))
        for s in range(chunk):
            t = c0 + s
            if t % 8 == 0:   # logits from the oracle's own (bit-identical) observation of the state before step t
                ol_pop = OP.mlp_logits(pop, o_pop.reshape(n_ids * N, -1)).reshape(n_ids, N, -1)
                ol_gov = OP.mlp_logits(gov, o_gov.reshape(n_ids, -1))
                pl = pl_ring[s].reshape(E, N, g.A)[:n_ids].cpu().numpy()
                gl = gl_ring[s][:n_ids].cpu().numpy()
                worst = max(worst, check_logits(pl, ol_pop, "t=%d population logits" % t), check_logits(gl, ol_gov, "t=%d government logits" % t))
                if t % 40 == 0:
                    sel = list(range(0, n_ids, 9))
                    a_, t_ = check_samples(cfg["seed"], sel, N, [t] * len(sel), ol_pop[sel], ol_gov[sel], a_out[s][sel], g_out[s][sel],
                                           g.B, g.L, "t=%d" % t)
                    amb, tot = amb + a_, tot + t_
            _, _, o_pop, o_gov, o_rew, o_done = outs[s]
            compare_outputs(g, pop_obs[s], gov_obs[s], rew[s], done[s], o_pop, o_gov, o_rew, o_done, "config5 full size t=%d" % t)
        compare_state(g.get_state(0, n_ids), o.state(), "config5 full size state at t=%d" % (c0 + chunk))
    assert amb <= max(2, 0.01 * tot) and worst < 5e-3
    an = act_ring.cpu().numpy()
    assert an.min() >= 0 and an.max() < g.A


def test_masked_policy_rollout_teacher_forced():
    """f1 with the policy head: under ej_set_action_masking every sampled population
    action is available in the oracle's mask of the state before the step, is eps-consistent with
    the oracle's MASKED categorical, and the env never counts an invalid action."""
    import torch

    cfg = inputs.configs()["config5_policy"]
    N, R, E, T = cfg["N"], cfg["R"], 4, 48
    params = dict(cfg["params"], tax_period=16)
    pair = Pair(E, N, R, params, cfg["seed"])
    g = pair.g
    pop, gov = inputs.policy_weights(cfg, seed=3, std=0.3, bias_std=0.1)
    g.set_policy(pop, gov)
    g.set_action_masking(True)
    act_ring = torch.zeros((T, E, N), dtype=torch.int32, device="cuda")
    gov_ring = torch.zeros((T, E, g.B), dtype=torch.int32, device="cuda")
    pl_ring = torch.zeros((T, E * N, g.A), dtype=torch.float32, device="cuda")
    g.rollout(T, ring_depth=T, actions_ring=act_ring, gov_actions_ring=gov_ring, pop_logits_ring=pl_ring)
    torch.cuda.synchronize()
    a_out, g_out = act_ring.cpu().numpy(), gov_ring.cpu().numpy()
    pl = pl_ring.cpu().numpy().reshape(T, E, N, -1)
    o_pop, o_gov = pair.o[0].observe()
    amb = tot = masked_out = 0
    for t in range(T):
        mask = pair.o[0].action_mask()
        masked_out += int((mask == 0).sum())
        ol_pop = OP.mlp_logits(pop, o_pop.reshape(E * N, -1)).reshape(E, N, -1)
        check_logits(pl[t], ol_pop, "t=%d population logits (reported unmasked)" % t)
        for e in range(E):
            for i in range(N):
                a = int(a_out[t, e, i])
                assert mask[e, i, a] == 1, "t=%d env %d agent %d: unavailable action %d sampled" % (t, e, i, a)
                if t % 6 == 0:
                    u = OP.philox_u(cfg["seed"], e, i, t, 0, 0)
                    assert OP.sample_consistent(ol_pop[e, i], u, a, EPS_CDF, mask[e, i]), "t=%d env %d agent %d action %d u=%g" % (t, e, i, a, u)
                    amb += OP.sample(ol_pop[e, i], u, mask[e, i]) != a
                    tot += 1
        o_pop, o_gov, _, _ = pair.o[0].step(a_out[t], g_out[t])
    compare_state(pair.g_state(), pair.o_state(), "masked policy rollout final state")
    assert masked_out > 0 and amb <= max(2, 0.01 * tot)
    assert sum(int(oracle.parse_state(w)["counters"][2]) for w in pair.g.get_state()) == 0
