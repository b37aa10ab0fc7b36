"""Small driver for compute-sanitizer (racecheck / memcheck): a few steps of ej_step, a short
ej_rollout with generated actions, a policy-driven rollout, masked sampling, factored observations and the section-5 variants, on shapes that exercise the
specialised kernel, the generic kernel and the book-cap path.  Not collected by pytest.

    compute-sanitizer --tool racecheck python tests/racecheck_driver.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch  # noqa: E402

from paper_2410_22165_b200 import binding, inputs  # noqa: E402


def run(name, E, steps, **over):
    cfg = inputs.configs()[name]
    params = dict(cfg["params"], **over)
    env = binding.Env(E, cfg["N"], cfg["R"], params)
    env.reset(3)
    acts, gov = inputs.action_stream(dict(cfg, params=params), steps, seed=3, E=E)
    for t in range(steps):
        env.step(torch.from_numpy(acts[t]).cuda(), torch.from_numpy(gov[t]).cuda())
    env.set_action_cdf(inputs.action_cdf(dict(cfg, params=params)))
    env.rollout(steps, ring_depth=2, obs_ring=env.new_obs(2), rew_ring=env.new_rew(2), done_ring=env.new_done(2))
    torch.cuda.synchronize()
    return env


if __name__ == "__main__":
    run("tiny_dense", 2, 12)
    run("config2_paper", 2, 12, tax_period=5)
    run("config3_resources", 1, 6, tax_period=3)
    run("config4_population", 1, 4, tax_period=2)
    cfg = inputs.configs()["config5_policy"]
    env = run("config5_policy", 2, 4, tax_period=3)
    env.set_policy(*inputs.policy_weights(cfg, seed=1, std=0.3))
    env.rollout(4)
    env.set_action_masking(True)   # f1: masked policy sampler, mask kernel, masked table generator
    env.rollout(3)
    env.action_mask()
    env2 = run("config2_paper", 2, 3)
    env2.set_action_masking(True)
    env2.rollout(6)
    # f2 / f3: factored rings, growing skills, normal skill init, the section-5 kernel variants, host factored step
    for name, E in (("section5_r4", 2), ("section5_r12", 1)):
        env3 = run(name, E, 5)
        c3 = inputs.configs()[name]
        if name == "section5_r4":
            priv, shared, govr = env3.new_factored_obs(2)
            env3.rollout(4, ring_depth=2, obs_priv_ring=priv, obs_shared_ring=shared, obs_gov_ring=govr)
            a3, g3 = inputs.action_stream(c3, 2, seed=4, E=E)
            hp = np.zeros((E, c3["N"], env3.D_priv), np.float32)
            hs = np.zeros((E, env3.D_shared_pad), np.float32)
            for t in range(2):
                env3.step_host_factored(a3[t], g3[t], hp, hs)
    run("config2_paper", 2, 6, tax_period=3, skill_growth_rate=0.005, skill_max=5.0)
    torch.cuda.synchronize()
    print("driver done")
