"""GPU parity tests: the CUDA path, called through the C ABI, against the CPU oracle on the same
seeded inputs (sizes the oracle finishes in seconds, spanning several CTAs / warps and ragged
tails), plus the edge cases of the method.  Run on the B200 box: ``pytest -m gpu``."""
import numpy as np
import pytest

import oracle
from conftest import Act
from paper_2410_22165_b200 import inputs
from parity import Pair, compare_outputs, compare_state, close, exact

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_cuda():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")


def run_episode(name, E, steps, seed=None, env_ids=None, state_every=1, **over):
    cfg = inputs.configs()[name]
    params = dict(cfg["params"], **over)
    seed = cfg["seed"] if seed is None else seed
    pair = Pair(E, cfg["N"], cfg["R"], params, seed, env_ids=env_ids)
    compare_state(pair.g_state(), pair.o_state(), "reset")
    acts, gov = inputs.action_stream(dict(cfg, params=params), steps, seed=seed, E=E)
    for t in range(steps):
        pair.step_and_compare(acts[t], gov[t], "%s t=%d" % (name, t), check_state=(t % state_every == 0 or t == steps - 1))
    return pair


def test_reset_and_observe_parity():
    for name, E in (("config1_tiny", 1), ("tiny_dense", 8), ("config2_paper", 5), ("config3_resources", 3)):
        cfg = inputs.configs()[name]
        pair = Pair(E, cfg["N"], cfg["R"], cfg["params"], 99)
        compare_state(pair.g_state(), pair.o_state(), name + " reset")
        pop, gov = pair.g.split_obs(pair.g.observe())
        o_pop, o_gov = pair.o[0].observe()
        exact(pop.cpu().numpy(), o_pop, name + " reset pop obs")
        close(gov.cpu().numpy(), o_gov, name + " reset gov obs")
        # observe must not disturb the state
        compare_state(pair.g_state(), pair.o_state(), name + " after observe")


def test_config1_tiny_full_episode():
    pair = run_episode("config1_tiny", 1, 55)  # 5 steps past the end: finished env is a no-op (G28)
    assert pair.g.get_state()[0, 0] == 50


@pytest.mark.parametrize("seed", [7, 1, 2])
def test_tiny_dense_full_episode(seed):
    pair = run_episode("tiny_dense", 8, 50, seed=seed)
    assert oracle.parse_state(pair.g.get_state()[0])["counters"][0] >= 0
    trades = sum(oracle.parse_state(w)["counters"][0] for w in pair.g.get_state())
    assert trades > 0


def test_config2_paper_scale_300_steps():
    pair = run_episode("config2_paper", 24, 300, state_every=7)
    s = oracle.parse_state(pair.g.get_state()[0])
    assert s["counters"][0] > 1000 and s["counters"][3] > 1000  # trades and expiries really happened


def test_config2_full_episode_few_envs():
    run_episode("config2_paper", 4, 1001, seed=1, state_every=50)


def test_config3_resources_parity():
    run_episode("config3_resources", 6, 250, state_every=10)


def test_config5_shape_parity():
    run_episode("config5_policy", 5, 200, state_every=10)


def test_config4_population_book_cap():
    pair = run_episode("config4_population", 2, 120, state_every=10)
    s = oracle.parse_state(pair.g.get_state()[0])
    assert max(len(b) for b in s["books"]) > 500  # the cap regime is reached


def test_per_resource_craft_mode():
    run_episode("tiny_dense", 6, 50, craft_mode=inputs.CRAFT_PER_RESOURCE)
    run_episode("config3_resources", 3, 120, craft_mode=inputs.CRAFT_PER_RESOURCE, state_every=10)


@pytest.mark.parametrize("N", [1, 2, 5, 31, 32, 33, 63, 97, 129, 250, 300, 417, 512, 600, 1024])
def test_ragged_population_sizes(N):
    cfg = dict(inputs.configs()["config2_paper"], N=N)
    params = dict(cfg["params"], tax_period=20, episode_length=80)
    pair = Pair(3, N, 2, params, 5)
    acts, gov = inputs.action_stream(dict(cfg, params=params), 80, seed=5, E=3)
    for t in range(80):
        pair.step_and_compare(acts[t], gov[t], "N=%d t=%d" % (N, t), check_state=(t % 10 == 0 or t == 79))


def test_small_caps_and_short_expiry():
    # small per-agent cap, short expiry and a small book cap stress slot reuse and the FIFO pops
    run_episode("config2_paper", 6, 200, state_every=5, max_active_orders=3, order_expiry=4, book_cap=7, tax_period=25)
    run_episode("tiny_dense", 8, 50, max_active_orders=1, order_expiry=1)
    run_episode("tiny_dense", 8, 50, max_active_orders=32, order_expiry=100)


def test_invalid_and_out_of_range_actions():
    cfg = inputs.configs()["tiny_dense"]
    pair = Pair(4, cfg["N"], cfg["R"], cfg["params"], 3)
    rng = np.random.default_rng(0)
    A = pair.g.A
    for t in range(40):
        acts = rng.integers(-3, A + 3, size=(4, cfg["N"]), dtype=np.int32)
        gov = rng.integers(-2, 13, size=(4, pair.g.B), dtype=np.int32)
        pair.step_and_compare(acts, gov, "invalid t=%d" % t)
    s = oracle.parse_state(pair.g.get_state()[0])
    assert s["counters"][2] > 0 and s["counters"][4] > 0


def test_taxes_disabled_and_omega():
    run_episode("tiny_dense", 4, 50, taxes_enabled=0)
    run_episode("tiny_dense", 4, 50, omega=0.25, eta=0.5)


def test_paper_price_grid_and_defaults():
    # Table 2 defaults as printed: prices [2,4,6,8,10], 3 brackets [50;100], U[0,1) skills
    p = inputs.default_params()
    p.update(episode_length=120, tax_period=30)
    cfg = dict(E=5, N=20, R=2, T=120, seed=4, action_mix="uniform", params=p)
    pair = Pair(5, 20, 2, p, 4)
    acts, gov = inputs.action_stream(cfg, 120, seed=4, E=5)
    for t in range(120):
        pair.step_and_compare(acts[t], gov[t], "defaults t=%d" % t, check_state=(t % 10 == 0))


@pytest.mark.parametrize("N,R,prices", [(100, 4, [3, 6, 9]), (100, 2, [2, 4, 6, 8, 10]), (100, 12, [3, 6, 9]), (60, 5, list(range(1, 11))),
                                        (1000, 3, [3, 6, 9])])
def test_shapes_of_generic_and_specialised_kernels(N, R, prices):
    # the step kernel has shape-specialised variants (R, P compile-time) for BASELINE.json's shapes and a
    # generic one for everything else: the paper's section-5 shapes (r = 4 and r = 12 with prices {3,6,9}:
    # 30 and 86 actions) and other odd shapes run the generic kernel, [2..10] at R = 2 a specialised one
    p = inputs.default_params()
    p.update(prices=prices, episode_length=60, tax_period=20, thresholds=inputs.THRESHOLDS_7, skill_init=inputs.SKILL_PARETO_CLIP,
             craft_distinct=2)
    E = 2 if N == 1000 else 4
    cfg = dict(E=E, N=N, R=R, T=60, seed=9, action_mix="uniform", params=p)
    pair = Pair(E, N, R, p, 9)
    if R in (4, 12) and len(prices) == 3:
        assert pair.g.A == {4: 30, 12: 86}[R]
    acts, gov = inputs.action_stream(cfg, 60, seed=9, E=E)
    for t in range(60):
        pair.step_and_compare(acts[t], gov[t], "shape N=%d R=%d P=%d t=%d" % (N, R, len(prices), t), check_state=(t % 10 == 0 or t == 59))


# ---------------- f3: skill growth (G41) ----------------
GROWTH = dict(skill_growth_rate=0.005, skill_max=5.0)


def test_skill_growth_step_parity():
    # uniform skills in [0,1) grow toward 5; Pareto skills clipped to [1,10] start partly ABOVE the maximum, where the
    # damped bonus is negative until the cap applies: both branches of the rule, state (skills included) bit-exact
    grown = run_episode("tiny_dense", 6, 50, **GROWTH)
    fixed = run_episode("tiny_dense", 6, 50)
    assert (grown.g_state() != fixed.g_state()).any(), "growth left the skills unchanged"
    run_episode("config2_paper", 5, 220, state_every=20, **GROWTH)
    run_episode("config3_resources", 3, 120, state_every=10, craft_mode=inputs.CRAFT_PER_RESOURCE, **GROWTH)
    run_episode("config2_paper", 3, 150, state_every=25, skill_growth_rate=0.25, skill_max=2.0)


@pytest.mark.parametrize("R", [4, 12])
def test_skill_growth_section5_shapes(R):
    # the paper's section-5 workload: r = 4 / 12 resources, prices {3,6,9}, skills that grow
    p = inputs.default_params()
    p.update(prices=[3, 6, 9], episode_length=80, tax_period=20, thresholds=inputs.THRESHOLDS_7, craft_distinct=2, **GROWTH)
    cfg = dict(E=4, N=100, R=R, T=80, seed=11, action_mix="uniform", params=p)
    pair = Pair(4, 100, R, p, 11)
    acts, gov = inputs.action_stream(cfg, 80, seed=11, E=4)
    for t in range(80):
        pair.step_and_compare(acts[t], gov[t], "growth R=%d t=%d" % (R, t), check_state=(t % 10 == 0 or t == 79))


def test_normal_skill_init_and_section5_workload():
    # EJ_SKILL_NORMAL_CLIP at reset (bit-exact skills), then the section-5 presets through the persistent rollout
    for name, E in (("section5_r4", 5), ("section5_r12", 3)):
        cfg = inputs.configs()[name]
        pair = Pair(E, cfg["N"], cfg["R"], cfg["params"], 21)
        assert pair.g.A == {4: 30, 12: 86}[cfg["R"]]                             # P:350, read from ej_layout
        assert pair.g.noop_action == pair.g.A - 1 and pair.g.base_buy == cfg["R"] + 1 and pair.g.D_pop == 6 + 8 * cfg["R"] + 3
        compare_state(pair.g_state(), pair.o_state(), name + " reset")
        sk = np.concatenate([oracle_skills(w) for w in pair.g_state()])
        assert sk.min() >= 0.0 and sk.max() <= 5.0 and 0.9 < sk.mean() < 1.25 and (sk == 0.0).mean() > 0.1
        _rollout_vs_oracle(name, E, 90)
    _rollout_vs_oracle("section5_r4", 4096, 50, env_ids=[0, 1999, 4095], ring=2)
    _rollout_vs_oracle("section5_r12", 2048, 40, env_ids=[0, 2047], ring=2)
    run_episode("tiny_dense", 4, 50, skill_init=inputs.SKILL_NORMAL_CLIP, skill_mean=2.0, skill_std=0.5, skill_clip_lo=0.25,
                skill_clip_hi=3.0)


def oracle_skills(words):
    from oracle import parse_state
    s = parse_state(words)
    return np.concatenate([np.asarray(s["SG"], np.float64).ravel(), np.asarray(s["SC"], np.float64).ravel()])


def test_skill_growth_rollout_and_bad_params():
    from paper_2410_22165_b200 import binding

    _rollout_vs_oracle("config2_paper", 6, 130, **GROWTH)
    _rollout_vs_oracle("headline", 4096, 60, env_ids=[0, 2049, 4095], ring=2, **GROWTH)
    cfg = inputs.configs()["config1_tiny"]
    for bad in (dict(skill_growth_rate=-0.1, skill_max=5.0), dict(skill_growth_rate=0.005, skill_max=0.0)):
        with pytest.raises(binding.EjError):
            binding.Env(1, cfg["N"], cfg["R"], dict(cfg["params"], **bad))


# ---------------- scripted worked examples, seeded into the GPU through the canonical dump ----------------
def _scripted(N, R, params, setup, steps):
    """setup(oracle_env) scripts the oracle; its dump is loaded into the GPU env; both then step."""
    pair = Pair(1, N, R, params, 0)
    setup(pair.o[0])
    pair.g.set_state(pair.o[0].get_state())
    compare_state(pair.g_state(), pair.o_state(), "after set_state")
    for k, (acts, gov) in enumerate(steps):
        pair.step_and_compare(np.array(acts, np.int32), np.array(gov, np.int32), "scripted step %d" % k)
    return pair


def test_scripted_tax_example(small_params):
    # income 130 at (10%,30%,50%) on [50;100] pays 35; n = 2 redistribution
    a = Act(1, 10)
    p = dict(small_params, starting_coin=0.0, tax_period=2, episode_length=10, craft_units=1, craft_distinct=1)

    def setup(o):
        o.set_agent(0, 0, 0.0, inv=[1], SG=[0.0], SC=13.0)
        o.set_rates(0, [np.float32(0.1), np.float32(0.3), np.float32(0.5)])

    pair = _scripted(2, 1, p, setup, [([[a.craft(), a.noop]], [[2, 6, 10]]), ([[a.noop, a.noop]], [[1, 2, 3]])])
    s = oracle.parse_state(pair.g.get_state()[0])
    assert s["coin"].tolist() == [130.0 - 35.0 + 17.5, 17.5] and s["income"].tolist() == [0.0, 0.0]


def test_scripted_trade_price_of_last_placed(small_params):
    a = Act(2, 10)
    p = dict(small_params, starting_coin=15.0)

    def setup(o):
        o.set_agent(0, 1, 15.0, inv=[1, 0])

    pair = _scripted(2, 2, p, setup, [([[a.noop, a.sell(0, 3)]], [[0, 0, 0]]), ([[a.buy(0, 5), a.noop]], [[0, 0, 0]])])
    s = oracle.parse_state(pair.g.get_state()[0])
    assert s["coin"].tolist() == [9.0, 21.0] and s["last_price"].tolist() == [6, 0]  # price of the later order
    pair = _scripted(2, 2, p, setup, [([[a.buy(0, 7), a.noop]], [[0, 0, 0]]), ([[a.noop, a.sell(0, 4)]], [[0, 0, 0]])])
    s = oracle.parse_state(pair.g.get_state()[0])
    assert s["coin"].tolist() == [10.0, 20.0] and s["last_price"][0] == 5


def test_scripted_expiry_boundary(small_params):
    a = Act(1, 10)
    p = dict(small_params, starting_coin=15.0, order_expiry=30, episode_length=100, tax_period=100, craft_distinct=1)
    steps = [([[a.buy(0, 5)]], [[0, 0, 0]])] + [([[a.noop]], [[0, 0, 0]])] * 30
    pair = _scripted(1, 1, p, lambda o: None, steps)
    s = oracle.parse_state(pair.g.get_state()[0])
    assert s["n_live"][0] == 0 and s["coin"][0] == 15.0 and s["counters"][3] == 1


def test_set_state_round_trip_mid_episode():
    cfg = inputs.configs()["config2_paper"]
    pair = run_episode("config2_paper", 3, 60, state_every=20)
    w = pair.g.get_state()
    from paper_2410_22165_b200 import binding
    g2 = binding.Env(3, cfg["N"], cfg["R"], cfg["params"])
    g2.reset(cfg["seed"])
    g2.set_state(w)
    exact(g2.get_state()[:, :11], w[:, :11], "round trip header")
    exact(g2.get_state()[:, 13:], w[:, 13:], "round trip body")
    # both continue identically
    import torch
    acts, gov = inputs.action_stream(cfg, 30, seed=77, E=3)
    for t in range(30):
        a, g = torch.from_numpy(acts[t]).cuda(), torch.from_numpy(gov[t]).cuda()
        o1, r1, d1 = pair.g.step(a, g)
        o2, r2, d2 = g2.step(a, g)
        assert torch.equal(o1, o2) and torch.allclose(r1, r2, rtol=1e-5, atol=1e-6) and torch.equal(d1, d2)
    exact(g2.get_state()[:, 13:], pair.g.get_state()[:, 13:], "round trip continuation")


# ---------------- persistent rollout ----------------
def _rollout_vs_oracle(name, E, T, env_ids=None, supplied_actions=False, ring=None, **over):
    import torch

    cfg = inputs.configs()[name]
    params = dict(cfg["params"], **over)
    pair = Pair(E, cfg["N"], cfg["R"], params, cfg["seed"], env_ids=env_ids)
    g = pair.g
    cdf = inputs.action_cdf(dict(cfg, params=params))
    g.set_action_cdf(cdf)
    depth = T if ring is None else ring
    obs_ring, rew_ring, done_ring = g.new_obs(depth), g.new_rew(depth), g.new_done(depth)
    act_ring = torch.zeros((depth, E, cfg["N"]), dtype=torch.int32, device="cuda")
    gov_ring = torch.zeros((depth, E, g.B), dtype=torch.int32, device="cuda")
    kw = {}
    if supplied_actions:
        acts, gov = inputs.action_stream(dict(cfg, params=params), T, seed=5, E=E)
        kw = dict(actions_in=torch.from_numpy(acts).cuda(), gov_actions_in=torch.from_numpy(gov).cuda())
    g.rollout(T, ring_depth=depth, obs_ring=obs_ring, rew_ring=rew_ring, done_ring=done_ring, actions_ring=act_ring,
              gov_actions_ring=gov_ring, **kw)
    torch.cuda.synchronize()
    pop, gv = g.split_obs(obs_ring)
    pop, gv, rew, done = pop.cpu().numpy(), gv.cpu().numpy(), rew_ring.cpu().numpy(), done_ring.cpu().numpy()
    a_out, g_out = act_ring.cpu().numpy(), gov_ring.cpu().numpy()
    ids = pair.env_ids
    for t in range(T):
        if supplied_actions:
            o_a, o_g = acts[t][ids], gov[t][ids]
        else:
            o_a, o_g = pair.o_draw(cdf)
        slot = t % depth
        if t >= T - depth:  # still in the ring
            exact(a_out[slot][ids], o_a, "rollout actions t=%d" % t)
            exact(g_out[slot][ids], o_g, "rollout gov actions t=%d" % t)
        if pair.full:
            o_pop, o_gov, o_rew, o_done = pair.o[0].step(o_a, o_g)
        else:
            outs = [o.step(o_a[k:k + 1], o_g[k:k + 1]) for k, o in enumerate(pair.o)]
            o_pop, o_gov, o_rew, o_done = (np.concatenate([x[j] for x in outs]) for j in range(4))
        if t >= T - depth:
            compare_outputs(g, pop[slot][ids], gv[slot][ids], rew[slot][ids], done[slot][ids], o_pop, o_gov, o_rew, o_done,
                            "rollout %s t=%d" % (name, t))
    compare_state(pair.g_state(), pair.o_state(), "rollout final state")
    return pair


def test_rollout_generated_actions_tiny():
    _rollout_vs_oracle("tiny_dense", 8, 50)
    _rollout_vs_oracle("config1_tiny", 1, 50)


def test_rollout_generated_actions_paper_scale():
    _rollout_vs_oracle("config2_paper", 12, 150)


def test_rollout_supplied_actions_and_small_ring():
    _rollout_vs_oracle("config2_paper", 6, 100, supplied_actions=True, ring=4)


def test_rollout_config4_market_mix():
    _rollout_vs_oracle("config4_population", 2, 60)


def test_rollout_in_two_calls_equals_one_call():
    import torch
    from paper_2410_22165_b200 import binding

    cfg = inputs.configs()["config2_paper"]
    a = binding.Env(7, cfg["N"], cfg["R"], cfg["params"])
    b = binding.Env(7, cfg["N"], cfg["R"], cfg["params"])
    a.reset(3)
    b.reset(3)
    a.rollout(120)
    b.rollout(50)
    b.rollout(70)
    torch.cuda.synchronize()
    assert (a.get_state() == b.get_state()).all()


def test_full_size_headline_sampled_envs():
    """BASELINE.json's headline launch configuration (E=4096, N=100, R=2) as bench.py runs it;
    sampled envs are re-computed one by one by the oracle (keyed by global env id)."""
    ids = [0, 1, 147, 148, 2367, 2368, 4094, 4095]
    _rollout_vs_oracle("headline", 4096, 130, env_ids=ids, ring=2)


def test_full_size_config3_and_config4_sampled_envs():
    _rollout_vs_oracle("config3_resources", 4096, 110, env_ids=[0, 2047, 4095], ring=2)
    _rollout_vs_oracle("config4_population", 256, 40, env_ids=[0, 255], ring=2)


def test_results_do_not_depend_on_batch_or_env_id_base():
    import torch
    from paper_2410_22165_b200 import binding

    cfg = inputs.configs()["tiny_dense"]
    big = binding.Env(6, cfg["N"], cfg["R"], cfg["params"])
    one = binding.Env(1, cfg["N"], cfg["R"], dict(cfg["params"], env_id_base=4))
    big.reset(5)
    one.reset(5)
    big.rollout(40)
    one.rollout(40)
    torch.cuda.synchronize()
    assert (big.get_state(4, 1) == one.get_state()).all()


def test_error_paths():
    from paper_2410_22165_b200 import binding

    p = inputs.default_params()
    with pytest.raises(binding.EjError) as ei:
        binding.Env(1, 4, 2, dict(p, prices=[2, 2, 3]))
    assert ei.value.code == binding.EJ_ERR_PARAM and "prices" in str(ei.value)
    with pytest.raises(binding.EjError) as ei:
        binding.Env(1, 4, 2, dict(p, eta=1.0))
    assert "eta" in str(ei.value)
    with pytest.raises(binding.EjError) as ei:
        binding.Env(1, 2000, 2, p)
    assert "N" in str(ei.value)
    env = binding.Env(1, 4, 2, p)
    import torch
    with pytest.raises(binding.EjError) as ei:
        env.step(torch.zeros((1, 4), dtype=torch.int32, device="cuda"), torch.zeros((1, 3), dtype=torch.int32, device="cuda"))
    assert ei.value.code == binding.EJ_ERR_STATE


@pytest.mark.parametrize("name", ["config2_paper", "tiny_dense", "config3_resources", "config4_population"])
def test_government_statistics_on_adversarial_states(name):
    """a10 on states the episodes never reach: inventories from 0 to 60,000 (the 64-bit sum path of
    the integer metrics), all-equal and two-valued populations, and jumps between rounds so that the
    median hints kept from the previous call are useless (walk-select gives up -> bitwise search /
    sorting network).  Each round: oracle state -> ej_set_state -> ej_observe, then one no-op step."""
    import torch

    cfg = inputs.configs()[name]
    E, N, R = 2, cfg["N"], cfg["R"]
    params = dict(cfg["params"], episode_length=1000)
    pair = Pair(E, N, R, params, 11)
    rng = np.random.default_rng(5)
    A = pair.g.A
    shapes = ["wide", "equal", "two", "small", "huge", "zero", "wide"]
    for rnd, shape in enumerate(shapes):
        for e in range(E):
            for i in range(N):
                if shape == "wide":
                    inv = rng.integers(0, 3000, R)
                    coin = float(np.float32(rng.uniform(0, 5000)))
                elif shape == "equal":
                    inv, coin = np.full(R, 7), 12.5
                elif shape == "two":
                    inv, coin = np.where(rng.random(R) < 0.5, 1, 50000), float(rng.choice([0.0, 1e4]))
                elif shape == "small":
                    inv, coin = rng.integers(0, 4, R), float(np.float32(rng.uniform(0, 3)))
                elif shape == "huge":
                    inv, coin = rng.integers(4000, 60000, R), float(np.float32(rng.uniform(0, 1e5)))
                else:
                    inv, coin = np.zeros(R, np.int64), 0.0
                pair.o[0].set_agent(e, i, coin, [int(v) for v in inv], [1.0] * R, 1.0)
        pair.g.set_state(pair.o[0].get_state())
        pop, gov = pair.g.split_obs(pair.g.observe())
        o_pop, o_gov = pair.o[0].observe()
        exact(pop.cpu().numpy(), o_pop, "%s round %d (%s) pop obs" % (name, rnd, shape))
        close(gov.cpu().numpy(), o_gov, "%s round %d (%s) gov obs" % (name, rnd, shape))
        acts = np.full((E, N), A - 1, np.int32)  # everyone idles: the step kernel's statistics of the same state
        for rep in range(3):                     # (bucketed kernels: fall-back step, then steps on the renewed bounds)
            pair.step_and_compare(acts, np.zeros((E, pair.g.B), np.int32), "%s round %d (%s) noop step %d" % (name, rnd, shape, rep))


# ---------------- properties that hold at any size, checked on EVERY env of the full-size launches ----------------
def _check_invariants_all_envs(name, steps):
    """Full-size rollout as bench.py launches it; parity.check_dump_invariants on the dump of all E envs."""
    import torch
    from paper_2410_22165_b200 import binding
    from parity import check_dump_invariants

    cfg = inputs.configs()[name]
    E = cfg["E"]
    env = binding.Env(E, cfg["N"], cfg["R"], cfg["params"])
    env.reset(cfg["seed"])
    env.set_action_cdf(inputs.action_cdf(cfg))
    env.rollout(steps)
    torch.cuda.synchronize()
    w = np.concatenate([env.get_state(b, min(512, E - b)) for b in range(0, E, 512)])   # int32 [E][state_words]
    assert w.shape[0] == E
    check_dump_invariants(w, cfg, steps)
    trades = w[:, 6]
    assert (trades > 0).mean() > 0.99                                                 # the workload really trades
    assert len(np.unique(w[:, 6:11], axis=0)) > E // 4                                # envs are keyed by their id


def test_full_size_invariants_on_every_env_headline():
    _check_invariants_all_envs("headline", 75)


def test_full_size_invariants_on_every_env_other_workloads():
    _check_invariants_all_envs("config3_resources", 45)
    _check_invariants_all_envs("section5_r4", 45)
    _check_invariants_all_envs("section5_r12", 40)
    _check_invariants_all_envs("config4_population", 35)     # N = 1000, book cap K = N (G15)
