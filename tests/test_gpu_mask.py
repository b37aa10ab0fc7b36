"""f1 parity: ej_action_mask (CUDA) against orc_action_mask (oracle), byte for byte, on states the
two reach by the same (bit-exact) trajectory.  P:197-200."""
import numpy as np
import pytest

from paper_2410_22165_b200 import inputs

pytestmark = pytest.mark.gpu


def _run(name, E, steps, every, params_over=None, seed=3):
    import torch
    from parity import Pair

    cfg = inputs.configs()[name]
    params = dict(cfg["params"], **(params_over or {}))
    pair = Pair(E, cfg["N"], cfg["R"], params, seed)
    acts, gov = inputs.action_stream(dict(cfg, params=params), steps, seed=seed, E=E)
    A = pair.g.A
    m0 = pair.g.action_mask().cpu().numpy()
    assert np.array_equal(m0, pair.o[0].action_mask()), "mask of the reset state"
    seen0 = seen1 = 0
    for t in range(steps):
        pair.step_and_compare(acts[t] % A, gov[t], "%s t=%d" % (name, t), check_state=False)
        if t % every == every - 1:
            mg = pair.g.action_mask()
            torch.cuda.synchronize()
            mg = mg.cpu().numpy()
            mo = pair.o[0].action_mask()
            assert mg.shape == mo.shape == (E, cfg["N"], A)
            bad = np.argwhere(mg != mo)
            assert bad.size == 0, "%s t=%d: %d mask bytes differ, first (env, agent, action) = %s" % (name, t, len(bad), bad[:1])
            seen0 += int((mo == 0).sum())
            seen1 += int((mo == 1).sum())
    assert seen0 > 0 and seen1 > 0  # both outcomes occur: the comparison is not vacuous


def test_mask_tiny_dense():
    _run("tiny_dense", 8, 50, 1)


def test_mask_tiny_per_resource_craft_and_low_cap():
    # E*N*A = 3*4*45 = 540 bytes per env row set: total not a multiple of the env stride in words
    _run("tiny_dense", 3, 50, 1, dict(craft_mode=1, max_active_orders=2))


def test_mask_paper_shape():
    _run("config2_paper", 5, 60, 10)


def test_mask_six_resources_odd_action_count():
    # PER_RESOURCE at R = 6: A = 133 (odd), so 4-byte output words straddle agents and envs
    _run("config3_resources", 3, 40, 10, dict(craft_mode=1))


def test_mask_full_size_sampled_envs():
    """Headline shape (E = 4096) in the launch configuration the bench uses; oracle on sampled envs."""
    import torch
    from parity import Pair

    cfg = inputs.configs()["headline"]
    E = cfg["E"]
    ids = [0, 1, 777, 2048, E - 1]
    pair = Pair(E, cfg["N"], cfg["R"], cfg["params"], cfg["seed"], env_ids=ids)
    pair.g.set_action_cdf(inputs.action_cdf(cfg))
    pair.g.rollout(40)
    cdf = inputs.action_cdf(cfg)
    for o in pair.o:
        for t in range(40):
            a, g = o.draw_actions(cdf)
            o.step(a, g, want_obs=False)
    mg = pair.g.action_mask()
    torch.cuda.synchronize()
    mg = mg.cpu().numpy()
    for o, e in zip(pair.o, ids):
        assert np.array_equal(mg[e], o.action_mask()[0]), "env %d" % e
    # structure that holds at any size: gather and no-op columns are all ones
    assert mg[:, :, : cfg["R"]].all() and mg[:, :, -1].all()


def test_mask_errors():
    from paper_2410_22165_b200 import binding

    cfg = inputs.configs()["tiny_dense"]
    env = binding.Env(2, cfg["N"], cfg["R"], cfg["params"])
    with pytest.raises(binding.EjError):
        binding.ej_action_mask(env.h, None)  # NULL pointer
    env.reset(1)
    m = env.action_mask()
    with pytest.raises(binding.EjError):
        binding.ej_action_mask(env.h, m.data_ptr() + 1)  # misaligned


# ---- f1 masked sampling: the rollout's table generator under the mask ----

def _masked_rollout(name, E, steps, params_over=None, seed=6, env_ids=None, mix=None):
    import torch
    from parity import Pair, compare_state

    cfg = inputs.configs()[name]
    params = dict(cfg["params"], **(params_over or {}))
    pair = Pair(E, cfg["N"], cfg["R"], params, seed, env_ids=env_ids)
    cdf = inputs.action_cdf(cfg if mix is None else dict(inputs.configs()[mix], R=cfg["R"], params=params))
    pair.g.set_action_cdf(cdf)
    pair.g.set_action_masking(True)
    depth = steps
    actions_ring = torch.zeros((depth, E, cfg["N"]), dtype=torch.int32, device="cuda")
    pair.g.rollout(steps, ring_depth=depth, actions_ring=actions_ring)
    torch.cuda.synchronize()
    got = actions_ring.cpu().numpy()
    ids = pair.env_ids
    for t in range(steps):
        for o, e in zip(pair.o, ids) if env_ids is not None else [(pair.o[0], None)]:
            a, g = o.draw_actions(cdf, masked=True)
            want = got[t] if e is None else got[t, e:e + 1]
            assert np.array_equal(a, want), "%s t=%d env %s: masked draws differ" % (name, t, e)
            o.step(a, g, want_obs=False)
    compare_state(pair.g_state(), pair.o_state(), name + " masked rollout")
    return pair


def test_masked_rollout_tiny():
    pair = _masked_rollout("tiny_dense", 8, 50)
    import oracle
    assert sum(int(oracle.parse_state(w)["counters"][2]) for w in pair.g.get_state()) == 0  # no invalid action


def test_masked_rollout_tiny_per_resource_low_cap_mixed_table():
    _masked_rollout("tiny_dense", 5, 50, dict(craft_mode=1, max_active_orders=2), mix="config4_population")


def test_masked_rollout_paper_shape_specialised_kernel():
    import oracle
    pair = _masked_rollout("config2_paper", 6, 120)
    assert sum(int(oracle.parse_state(w)["counters"][2]) for w in pair.g.get_state()) == 0


def test_masked_rollout_six_resources():
    _masked_rollout("config3_resources", 3, 60)


def test_masked_rollout_full_size_sampled_envs():
    cfg = inputs.configs()["headline"]
    _masked_rollout("headline", cfg["E"], 40, env_ids=[0, 1500, cfg["E"] - 1], seed=cfg["seed"])


def test_masked_rollout_section5_growing_skills():
    # the paper's section-5 workload as its agents meet it: masked draws over 30 / 86 actions while the
    # skills grow; the mask of the reached state, byte for byte
    import oracle
    import torch
    for name, E in (("section5_r4", 4), ("section5_r12", 2)):
        pair = _masked_rollout(name, E, 70)
        assert sum(int(oracle.parse_state(w)["counters"][2]) for w in pair.g.get_state()) == 0
        mg = pair.g.action_mask()
        torch.cuda.synchronize()
        assert np.array_equal(mg.cpu().numpy(), pair.o[0].action_mask()), name
