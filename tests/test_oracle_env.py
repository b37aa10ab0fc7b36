"""Environment-level pins of the oracle: scripted worked examples, statistical pins of the
keyed draws, and the invariants of SURVEY.md section 4(2) on fuzzed episodes.  CPU only."""
import numpy as np
import pytest

import oracle
from conftest import Act
from paper_2410_22165_b200 import inputs


def make(E, N, R, params, seed=0):
    env = oracle.OracleEnv(E, N, R, params)
    env.reset(seed)
    return env


def st(env, e=0):
    return oracle.parse_state(env.get_state(e, 1)[0])


def gov0(env, n=1):
    return np.zeros((n, env.B), np.int32)


# ---------------- scripted worked examples ----------------
def test_reset_state(small_params):
    p = dict(small_params, starting_coin=15.0)
    env = make(3, 5, 2, p, seed=7)
    for e in range(3):
        s = st(env, e)
        assert s["t"] == 0 and (s["coin"] == 15.0).all()
        assert not s["inv"].any() and not s["esc_coin"].any() and not s["esc_res"].any()
        assert (s["labor"] == 0).all() and (s["income"] == 0).all() and (s["rates"] == 0).all()
        assert all(len(b) == 0 for b in s["books"])
        assert ((s["SG"] >= 0) & (s["SG"] < 1)).all() and ((s["SC"] >= 0) & (s["SC"] < 1)).all()
    obs_pop, obs_gov = env.observe()
    assert obs_pop.shape == (3, 5, 6 + 8 * 2 + 3) and obs_gov.shape == (3, 3 * 5 + 3 + 2)
    assert np.allclose(obs_pop[:, :, 0], 0.15)
    env2 = make(3, 5, 2, p, seed=7)
    assert (env.get_state() == env2.get_state()).all()
    env3 = make(3, 5, 2, p, seed=8)
    assert (env.get_state() != env3.get_state()).any()


def test_escrow_examples_and_order_cap(small_params):
    a = Act(2, 10)
    p = dict(small_params, starting_coin=15.0, max_active_orders=15)
    env = make(1, 2, 2, p)
    env.set_agent(0, 1, 0.0, inv=[0, 1])
    # buy r0 at 6 with coin 15 -> coin 9, escrow 6; sell r1 with 1 unit -> inventory 0, escrow 1
    env.step([[a.buy(0, 5), a.sell(1, 9)]], gov0(env))
    s = st(env)
    assert s["coin"][0] == 9.0 and s["esc_coin"][0] == 6 and s["n_live"][0] == 1
    assert s["inv"][1, 1] == 0 and s["esc_res"][1, 1] == 1 and s["n_live"][1] == 1
    assert s["books"][0].tolist() == [[6, 0, 0]] and s["books"][3].tolist() == [[10, 1, 0]]
    assert s["labor"][0] == np.float32(0.05) and s["labor"][1] == np.float32(0.05)
    # an agent that cannot pay / has no unit: invalid, nothing changes, no labor (G2)
    before = env.get_state().copy()
    env.step([[a.buy(0, 9), a.sell(0, 0)]], gov0(env))
    s2 = st(env)
    assert s2["counters"][2] == 2 and s2["coin"][0] == 9.0 and s2["labor"][0] == np.float32(0.05)
    assert (env.get_state()[0, 13:] == before[0, 13:]).all()
    # 16th order with cap 15 is rejected
    env = make(1, 1, 1, dict(p, starting_coin=100.0, craft_distinct=1))
    for k in range(16):
        env.step([[Act(1, 10).buy(0, 0)]], gov0(env))
    s = st(env)
    assert s["n_live"][0] == 15 and s["esc_coin"][0] == 15 and s["coin"][0] == 85.0 and s["counters"][2] == 1


def test_trade_settlement_last_placed_price(small_params):
    a = Act(2, 10)
    p = dict(small_params, starting_coin=15.0)
    env = make(1, 2, 2, p)
    env.set_agent(0, 1, 15.0, inv=[1, 0])
    env.step([[a.noop, a.sell(0, 3)]], gov0(env))        # ask r0@4 at t=0
    _, _, rew, _ = env.step([[a.buy(0, 5), a.noop]], gov0(env))  # bid r0@6 at t=1 -> trade at 6
    s = st(env)
    assert s["coin"].tolist() == [9.0, 21.0] and s["inv"].tolist() == [[1, 0], [0, 0]]
    assert not s["esc_coin"].any() and not s["esc_res"].any() and not s["n_live"].any()
    assert s["last_price"].tolist() == [6, 0] and s["income"].tolist() == [0.0, 6.0] and s["counters"][0] == 1
    # resting bid, later ask: price of the ask; buyer refunded the excess
    env = make(1, 2, 2, p)
    env.set_agent(0, 1, 15.0, inv=[1, 0])
    env.step([[a.buy(0, 7), a.noop]], gov0(env))          # bid@8 at t=0
    env.step([[a.noop, a.sell(0, 4)]], gov0(env))         # ask@5 at t=1 -> price 5, refund 3
    s = st(env)
    assert s["coin"].tolist() == [10.0, 20.0] and s["last_price"][0] == 5


def test_expiry_boundary(small_params):
    a = Act(1, 10)
    p = dict(small_params, starting_coin=15.0, order_expiry=30, episode_length=100, tax_period=100, craft_distinct=1)
    env = make(1, 1, 1, p)
    env.step([[a.buy(0, 5)]], gov0(env))                  # placed at t=0
    for t in range(1, 30):
        env.step([[a.noop]], gov0(env))
    s = st(env)                                           # after step t=29: still live
    assert s["t"] == 30 and s["n_live"][0] == 1 and s["coin"][0] == 9.0
    env.step([[a.noop]], gov0(env))                       # step t=30: 30 - 0 >= 30 -> removed, 6 coin back
    s = st(env)
    assert s["n_live"][0] == 0 and s["coin"][0] == 15.0 and s["esc_coin"][0] == 0 and s["counters"][3] == 1
    # an order still matches in its last round (G14): ask arrives at t=30
    env = make(1, 2, 1, p)
    env.set_agent(0, 1, 0.0, inv=[1])
    env.step([[a.buy(0, 5), a.noop]], gov0(env))
    for t in range(1, 30):
        env.step([[a.noop, a.noop]], gov0(env))
    env.step([[a.noop, a.sell(0, 0)]], gov0(env))
    s = st(env)
    assert s["counters"][0] == 1 and s["counters"][3] == 0 and s["coin"].tolist() == [14.0, 1.0]


def test_tax_collection_and_redistribution_example(small_params):
    # S:246 / P:195: income 130 at (10%,30%,50%) on [50;100], n=2: payer nets -35 + 17.5, other +17.5
    a = Act(1, 10)
    p = dict(small_params, starting_coin=0.0, tax_period=2, episode_length=10, craft_scale=10.0, craft_units=1,
             craft_distinct=1, thresholds=[50.0, 100.0])
    env = make(1, 2, 1, p)
    env.set_agent(0, 0, 0.0, inv=[1], SG=[0.0], SC=13.0)  # one craft pays 130
    env.set_rates(0, [np.float32(0.1), np.float32(0.3), np.float32(0.5)])
    env.step([[a.craft(), a.noop]], [[2, 6, 10]])         # t=0: craft, no boundary
    s = st(env)
    assert s["coin"].tolist() == [130.0, 0.0] and s["income"].tolist() == [130.0, 0.0]
    env.step([[a.noop, a.noop]], [[1, 2, 3]])             # t=1: (t+1)%2==0 -> collect, redistribute, new rates
    s = st(env)
    assert s["coin"].tolist() == [130.0 - 35.0 + 17.5, 17.5]
    assert s["income"].tolist() == [0.0, 0.0]
    assert s["rates"].tolist() == [np.float32(0.1), np.float32(0.2), np.float32(0.3)]  # table of 11 levels
    # tax is capped at the coin on hand (G17)
    env = make(1, 2, 1, p)
    env.set_agent(0, 0, 0.0, inv=[1], SG=[0.0], SC=13.0)
    env.set_rates(0, [1.0, 1.0, 1.0])
    env.step([[a.craft(), a.noop]], [[0, 0, 0]])
    env.set_agent(0, 0, 50.0, inv=[0], SG=[0.0], SC=13.0)  # spent 80 meanwhile
    env.step([[a.noop, a.noop]], [[0, 0, 0]])
    assert st(env)["coin"].tolist() == [25.0, 25.0]
    # out-of-range government level leaves that bracket's rate unchanged
    env.step([[a.noop, a.noop]], [[0, 0, 0]])
    env.step([[a.noop, a.noop]], [[5, 99, -1]])
    s = st(env)
    assert s["rates"].tolist() == [0.5, 0.0, 0.0] and s["counters"][4] == 2


def test_noop_step_and_done(small_params):
    a = Act(2, 10)
    p = dict(small_params, episode_length=3, tax_period=10)
    env = make(1, 3, 2, p)
    before = env.get_state()[0].copy()
    _, _, rew, done = env.step([[a.noop] * 3], gov0(env))
    after = env.get_state()[0]
    assert (rew == 0).all() and done[0] == 0 and after[0] == 1 and (after[1:] == before[1:]).all()
    env.step([[a.noop] * 3], gov0(env))
    _, _, _, done = env.step([[a.noop] * 3], gov0(env))
    assert done[0] == 1
    frozen = env.get_state()[0].copy()
    obs_pop, obs_gov, rew, done = env.step([[a.gather(0)] * 3], gov0(env))    # G28: no-op once done
    assert done[0] == 1 and (rew == 0).all() and (env.get_state()[0] == frozen).all()
    assert obs_pop[0, 0, -1] == 1.0


def test_observation_layout_and_market_stats(small_params):
    a = Act(2, 10)
    p = dict(small_params, starting_coin=15.0)
    env = make(1, 4, 2, p)
    env.set_agent(0, 2, 15.0, inv=[0, 2])
    env.set_agent(0, 3, 15.0, inv=[0, 1])
    # bids r0 {4, 8}, asks r1 {6, 9}: highest bid 8 / lowest ask 6, counts
    obs_pop, obs_gov, _, _ = env.step([[a.buy(0, 3), a.buy(0, 7), a.sell(1, 5), a.sell(1, 8)]], gov0(env))
    R, B = 2, 3
    o = obs_pop[0]
    assert o.shape == (4, 6 + 8 * R + B)
    f32 = np.float32
    assert o[0, 0] == f32(11.0) * f32(0.01) and o[1, 0] == f32(7.0) * f32(0.01)  # coin
    assert o[2, 1:3].tolist() == [0.0, f32(1) * f32(0.1)]                         # inventories
    assert o[0, 3] == f32(4) * f32(0.01)                                          # escrow coin
    assert o[2, 4:6].tolist() == [0.0, f32(0.1)]                                  # escrow units
    s = st(env)
    assert (o[:, 6:8] == s["SG"]).all() and (o[:, 8] == s["SC"]).all()
    assert (o[:, 9] == f32(0.05) * f32(0.01)).all()                               # labor
    m0 = [f32(8) * f32(0.1), 0.0, f32(2) * f32(0.1), 0.0, 0.0]
    m1 = [0.0, f32(6) * f32(0.1), 0.0, f32(2) * f32(0.1), 0.0]
    for i in range(4):
        assert o[i, 10:15].tolist() == m0 and o[i, 15:20].tolist() == m1
        assert o[i, 20:23].tolist() == [0.0, 0.0, 0.0]
        assert o[i, 23] == f32(1) / f32(10) and o[i, 24] == f32(1) / f32(50)     # timers (G27)
    g = obs_gov[0]
    assert g.shape == (3 * (3 + R) + B + 2,)
    coin = s["coin"].astype(np.float64)
    assert g[0] == pytest.approx(coin.mean() * 0.01, rel=1e-6) and g[1] == pytest.approx(coin.std() * 0.01, rel=1e-6)
    assert g[2] == np.median(s["coin"]) * f32(0.01)
    assert g[3 * 4 + 2] == np.median(s["inv"][:, 1].astype(np.float32)) * f32(0.1)


def test_government_row_hand_values(small_params):
    """Every entry of the government row (Fig.1, "mean, standard deviation, and median"; G26: metric
    order coin, labor, income, inv[r]; population std; each statistic times the metric's scale; then rates and
    the two timers, G27) on a 4-agent state built by scripted actions whose coin, labor, income and inventories
    all differ.  Scales are powers of two so that the hand values are exact in binary32."""
    import math

    a = Act(2, 10)
    p = dict(small_params, starting_coin=15.0, craft_units=1, craft_distinct=1, labor_craft=1.0, labor_trade=0.25,
             obs_scale_coin=0.5, obs_scale_labor=0.25, obs_scale_count=2.0, obs_scale_price=0.125)
    env = make(1, 4, 2, p)
    env.set_agent(0, 0, 15.0, inv=[3, 1], SC=1.25)
    env.set_agent(0, 1, 15.0, inv=[0, 5], SC=0.0)
    env.set_agent(0, 2, 15.0, inv=[7, 0], SC=0.0)
    env.set_agent(0, 3, 15.0, inv=[4, 2], SC=0.5)
    rates = [np.float32(0.1), np.float32(0.3), np.float32(0.5)]
    env.set_rates(0, rates)
    # step A: 0 crafts (pay 12.5), 1 bids 4 for r0, 2 idles, 3 crafts (pay 5)
    env.step([[a.craft(), a.buy(0, 3), a.noop, a.craft()]], gov0(env))
    # step B: 0 crafts again, 3 asks 3 for r0 -> trades with 1's bid at the later order's price 3
    _, g, _, _ = env.step([[a.craft(), a.noop, a.noop, a.sell(0, 2)]], gov0(env))
    s = st(env)
    assert s["coin"].tolist() == [40.0, 12.0, 15.0, 23.0]
    assert s["labor"].tolist() == [2.0, 0.25, 0.0, 1.25]
    assert s["income"].tolist() == [25.0, 0.0, 0.0, 8.0]
    assert s["inv"].tolist() == [[1, 1], [1, 5], [7, 0], [2, 2]]
    g = g[0]
    assert g.shape == (3 * (3 + 2) + 3 + 2,)
    f32 = np.float32
    want = [
        # coin, scale 0.5: mean 22.5, variance 473/4, median (15 + 23) / 2
        f32(22.5 * 0.5), f32(math.sqrt(118.25) * 0.5), f32(19.0 * 0.5),
        # labor, scale 0.25: mean 0.875, variance 2.5625/4, median (0.25 + 1.25) / 2
        f32(0.875 * 0.25), f32(math.sqrt(0.640625) * 0.25), f32(0.75 * 0.25),
        # income, scale 0.5 (a coin amount): mean 8.25, variance 416.75/4, median (0 + 8) / 2
        f32(8.25 * 0.5), f32(math.sqrt(104.1875) * 0.5), f32(4.0 * 0.5),
        # inventory of resource 0, scale 2: [1, 1, 7, 2]
        f32(2.75 * 2.0), f32(math.sqrt(6.1875) * 2.0), f32(1.5 * 2.0),
        # inventory of resource 1, scale 2: [1, 5, 0, 2]
        f32(2.0 * 2.0), f32(math.sqrt(3.5) * 2.0), f32(1.5 * 2.0),
    ]
    for k, w in enumerate(want):
        if k % 3 == 1:                                             # std: binary64 sqrt, one rounding to binary32
            assert abs(float(g[k]) - float(w)) <= 1.2e-7 * float(w), (k, g[k], w)
        else:
            assert g[k] == w, (k, g[k], w)
    assert g[15:18].tolist() == [float(r) for r in rates]          # the rates in force (set_rates), not the action
    assert g[18] == f32(2) / f32(10) and g[19] == f32(2) / f32(50)  # timers of t' = 2 (G27)
    # three agents (odd N): the median is the middle value, not a midpoint
    env3 = make(1, 3, 2, p)
    for i, (c, inv) in enumerate(((3.0, [9, 0]), (1.0, [2, 4]), (8.0, [5, 1]))):
        env3.set_agent(0, i, c, inv=inv, SC=0.0)
    _, g3 = env3.observe()
    assert g3[0, 2] == f32(3.0 * 0.5) and g3[0, 11] == f32(5 * 2.0) and g3[0, 14] == f32(1 * 2.0)
    assert g3[0, 0] == f32(4.0 * 0.5) and g3[0, 18] == 0.0 and g3[0, 19] == 0.0


def test_government_level_draws_recomputed_from_philox():
    """Rollout-mode government levels (G30): bracket b takes word b % 4 of Philox(ctr = (global env, N, t,
    stream 1 + b / 4), key = seed) and level = (x * L) >> 32.  Recomputed here from orc_philox4x32_10 (itself
    pinned by the Random123 known answers) for B = 7: two counter blocks, every word used once."""
    import ctypes as C

    L = oracle.lib()

    def philox(ctr, key):
        c, k, o = (C.c_uint32 * 4)(*ctr), (C.c_uint32 * 2)(*key), (C.c_uint32 * 4)()
        L.orc_philox4x32_10(c, k, o)
        return list(o)

    cfg = inputs.configs()["config2_paper"]
    seed = (0x9E3779B9 << 32) | 0x12345678                          # both key words matter
    N, nl = cfg["N"], len(cfg["params"]["rate_table"])
    env = make(3, N, 2, dict(cfg["params"], env_id_base=40), seed=seed)
    assert env.B == 7 and nl == 21
    cdf = inputs.action_cdf(cfg)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    seen = set()
    for t in range(6):
        acts, gov = env.draw_actions(cdf)
        for e in range(3):
            blocks = [philox([40 + e, N, t, 1], key), philox([40 + e, N, t, 2], key)]
            want = [(blocks[b // 4][b % 4] * nl) >> 32 for b in range(7)]
            assert gov[e].tolist() == want, (t, e)
            seen.update(want)
            # population action of agent i: smallest a with x0 < cdf[a] on stream 0 (word 0)
            for i in (0, 57, N - 1):
                x0 = philox([40 + e, i, t, 0], key)[0]
                assert acts[e, i] == int(np.searchsorted(cdf.astype(np.uint64), x0, side="right")) or \
                    (acts[e, i] == env.A - 1 and x0 >= cdf[-2])
        env.step(acts, gov, want_obs=False)
    assert len(seen) > 10                                          # the words differ: not one word for every bracket


def test_reward_is_utility_delta_and_gov_reward(small_params):
    a = Act(1, 10)
    p = dict(small_params, starting_coin=15.0, craft_units=1, craft_distinct=1)
    env = make(1, 2, 1, p)
    env.set_agent(0, 0, 15.0, inv=[1], SG=[0.0], SC=0.8)
    _, _, rew, _ = env.step([[a.craft(), a.gather(0)]], gov0(env))
    u = lambda c, l: (c ** 0.73 - 1) / 0.73 - l
    eta_err = 1e-6
    assert rew[0, 0] == pytest.approx(u(23.0, 1.0) - u(15.0, 0.0), abs=1e-5 + eta_err)   # +8 coin at SC=0.8
    assert rew[0, 1] == pytest.approx(-1.0, abs=1e-6)                                      # labor only
    # government: u_g = (1 - gini) * prod; before 30 (gini 0), after coins (23, 15): gini = (8+8)/(2*2*38)
    g = 16.0 / (2 * 2 * 38.0)
    assert rew[0, 2] == pytest.approx((1 - g) * 38.0 - 30.0, rel=1e-6)


# ---------------- statistical pins of the keyed draws ----------------
def test_gather_distribution_through_the_env():
    # T4 / S:79: P(>=1 | SG=0.5) = 0.6/1.1, P(=2 | SG=0.95) = 0.05/1.1, over 1e6 draws
    p = inputs.default_params()
    p.update(episode_length=500, tax_period=500, obs_scale_count=1.0, craft_distinct=1)
    N, T = 2000, 500
    env = make(1, N, 1, p, seed=11)
    half = N // 2
    for i in range(N):
        env.set_agent(0, i, 0.0, inv=[0], SG=[0.5 if i < half else 0.95], SC=0.0)
    prev = np.zeros(N)
    cnt1 = cnt2 = cnt0 = 0
    acts = np.zeros((1, N), np.int32)
    for t in range(T):
        obs_pop, _, _, _ = env.step(acts, gov0(env), want_obs=True)
        inv = obs_pop[0, :, 1].astype(np.float64)
        d = inv - prev
        prev = inv
        cnt1 += int((d[:half] >= 1).sum())
        cnt2 += int((d[half:] == 2).sum())
        cnt0 += int((d[half:] == 0).sum())
    n = half * T
    assert abs(cnt1 / n - 0.6 / 1.1) < 0.002
    assert abs(cnt2 / n - 0.05 / 1.1) < 0.001
    assert abs(cnt0 / n - 0.05 / 1.1) < 0.001


def test_pareto_skill_init_distribution():
    # T12: Pareto(alpha=4, x_m=1): P(x > s) = s^-4, mean 4/3
    p = inputs.default_params()
    p.update(skill_init=inputs.SKILL_PARETO_CLIP, skill_clip_lo=1.0, skill_clip_hi=1e9)
    env = make(200, 1000, 4, p, seed=5)
    sg = np.concatenate([oracle.parse_state(w)["SG"].ravel() for w in env.get_state()])
    sc = np.concatenate([oracle.parse_state(w)["SC"].ravel() for w in env.get_state()])
    x = np.concatenate([sg, sc]).astype(np.float64)
    n = len(x)
    assert n == 200 * 1000 * 5 and x.min() >= 1.0
    assert abs(x.mean() - 4.0 / 3.0) < 4 * np.sqrt(2.0 / 9.0 / n)
    for s in (1.5, 2.0, 3.0):
        q = s ** -4.0
        assert abs((x > s).mean() - q) < 5 * np.sqrt(q * (1 - q) / n)
    assert abs((x > 10).mean() - 1e-4) < 5e-5
    # different skills of one agent and different agents are different draws
    assert abs(np.corrcoef(sg.reshape(-1, 4)[:, 0], sg.reshape(-1, 4)[:, 1])[0, 1]) < 0.01
    # clipping (BASELINE.json: clipped to [1,10])
    p.update(skill_clip_hi=10.0)
    env = make(50, 1000, 4, p, seed=5)
    sg2 = np.concatenate([oracle.parse_state(w)["SG"].ravel() for w in env.get_state()])
    assert sg2.max() <= 10.0 and (sg2 == np.minimum(sg[:len(sg2)], 10.0)).all()


def test_uniform_skill_init_moments():
    p = inputs.default_params()
    env = make(100, 1000, 2, p, seed=3)
    x = np.concatenate([oracle.parse_state(w)["SG"].ravel() for w in env.get_state()]).astype(np.float64)
    assert 0 <= x.min() and x.max() < 1
    assert abs(x.mean() - 0.5) < 4 * np.sqrt(1 / 12 / len(x)) and abs(x.var() - 1 / 12) < 1e-3


def test_rollout_action_generator():
    cfgs = inputs.configs()
    cfg = cfgs["config2_paper"]
    env = make(4, 100, 2, cfg["params"], seed=9)
    cdf = inputs.action_cdf(cfg)
    counts = np.zeros(env.A)
    lv = np.zeros(21)
    acts0, gov0_ = env.draw_actions(cdf)
    acts1, _ = env.draw_actions(cdf)
    assert (acts0 == acts1).all()                                  # pure function of (seed, env, agent, t)
    for t in range(300):
        acts, gov = env.draw_actions(cdf)
        counts += np.bincount(acts.ravel(), minlength=env.A)
        lv += np.bincount(gov.ravel(), minlength=21)
        env.step(acts, gov, want_obs=False)
    n = counts.sum()
    assert np.abs(counts / n - 1 / env.A).max() < 5 * np.sqrt((1 / env.A) / n)
    assert np.abs(lv / lv.sum() - 1 / 21).max() < 5 * np.sqrt((1 / 21) / lv.sum())
    # config 4's mix: 70% market orders, price pmf of round(Normal(5,2)) clipped (BASELINE.json)
    cfg4 = cfgs["config4_population"]
    probs = inputs.action_probabilities(cfg4)
    assert probs.sum() == pytest.approx(1.0) and probs[3:43].sum() == pytest.approx(0.7)
    assert probs[3:13] / probs[3:13].sum() == pytest.approx(
        [.04006, .06559, .12098, .17467, .19741, .17467, .12098, .06559, .02783, .01222], abs=2e-5)
    env4 = make(1, 1000, 2, cfg4["params"], seed=9)
    cdf4 = inputs.action_cdf(cfg4)
    c4 = np.zeros(env4.A)
    for t in range(100):
        acts, gov = env4.draw_actions(cdf4)
        c4 += np.bincount(acts.ravel(), minlength=env4.A)
        env4.step(acts, gov, want_obs=False)
    assert np.abs(c4 / c4.sum() - probs).max() < 5 * np.sqrt(0.05 / c4.sum())


# ---------------- invariants on fuzzed episodes ----------------
def _totals(s):
    coin = s["coin"].astype(np.float64).sum() + s["esc_coin"].sum()
    res = s["inv"].sum(axis=0) + s["esc_res"].sum(axis=0)
    return coin, res


@pytest.mark.parametrize("name,E,steps", [("tiny_dense", 8, 50), ("config1_tiny", 1, 50), ("config2_paper", 2, 300),
                                          ("config3_resources", 1, 150)])
def test_invariants_on_fuzzed_episodes(name, E, steps):
    cfg = inputs.configs()[name]
    N, R, p = cfg["N"], cfg["R"], cfg["params"]
    a = Act(R, len(p["prices"]))
    env = make(E, N, R, p, seed=cfg["seed"])
    acts, gov = inputs.action_stream(cfg, steps, E=E)
    u0 = None
    ret = np.zeros((E, N))
    n_trades_seen = 0
    for t in range(steps):
        pre = [st(env, e) for e in range(E)]
        if u0 is None:
            u0 = [[oracle.lib().orc_utility(float(c), float(l), float(np.float32(p["eta"]))) for c, l in
                   zip(s["coin"], s["labor"])] for s in pre]
        _, _, rew, done = env.step(acts[t], gov[t])
        ret += rew[:, :N]
        for e in range(E):
            s0, s1 = pre[e], st(env, e)
            c0, r0 = _totals(s0)
            c1, r1 = _totals(s1)
            crafts = (acts[t, e] == a.craft())
            gathers = [(acts[t, e] == a.gather(r)) for r in range(R)]
            # escrow = sum of live orders, exactly; n_live = number of the agent's orders
            esc_coin = np.zeros(N, np.int64); esc_res = np.zeros((N, R), np.int64); live = np.zeros(N, np.int64)
            for b, book in enumerate(s1["books"]):
                for price, owner, placed in book:
                    live[owner] += 1
                    if b % 2 == 0:
                        esc_coin[owner] += price
                    else:
                        esc_res[owner, b // 2] += 1
                    assert 0 <= t - placed < p["order_expiry"]
                prices = book[:, 0] if len(book) else np.zeros(0)
                assert (np.diff(prices) <= 0).all() if b % 2 == 0 else (np.diff(prices) >= 0).all()
            assert (esc_coin == s1["esc_coin"]).all() and (esc_res == s1["esc_res"]).all()
            assert (live == s1["n_live"]).all() and live.max() <= p["max_active_orders"]
            # uncrossed book after matching
            for r in range(R):
                bb, ab = s1["books"][2 * r], s1["books"][2 * r + 1]
                if len(bb) and len(ab):
                    assert bb[0, 0] < ab[0, 0]
            # non-negativity
            assert (s1["coin"] >= 0).all() and (s1["inv"] >= 0).all() and (s1["labor"] >= s0["labor"]).all()
            # coin changes only by craft payouts; exact to fp32 rounding incl. tax boundaries (T8)
            made = sum(float(np.float32(s0["SC"][i]) * np.float32(p["craft_scale"])) for i in np.nonzero(crafts)[0]
                       if (s0["inv"][i] >= p["craft_units"]).sum() >= p["craft_distinct"])
            assert abs((c1 - c0) - made) < 1e-3 + N * 2.0 ** -21 + 2e-6 * c1
            # resources change only by gathering (+) and crafting (-units) (T8)
            for r in range(R):
                assert r1[r] - r0[r] <= 3 * 11 * gathers[r].sum()
                if not gathers[r].any() and not crafts.any():
                    assert r1[r] == r0[r]
            n_trades_seen = s1["counters"][0]
    # telescoping: sum of rewards = u_T - u_0
    for e in range(E):
        s = st(env, e)
        for i in range(N):
            uT = oracle.lib().orc_utility(float(s["coin"][i]), float(s["labor"][i]), float(np.float32(p["eta"])))
            assert ret[e, i] == pytest.approx(uT - u0[e][i], abs=2e-4 * steps ** 0.5 + 1e-6 * abs(uT))
    if name != "config1_tiny":
        assert n_trades_seen > 0


def test_all_zero_rates_equal_taxes_disabled():
    cfg = inputs.configs()["tiny_dense"]
    acts, gov = inputs.action_stream(cfg, 50, E=4)
    gov[:] = 0
    e1 = make(4, cfg["N"], cfg["R"], cfg["params"], seed=3)
    e2 = make(4, cfg["N"], cfg["R"], dict(cfg["params"], taxes_enabled=0), seed=3)
    for t in range(50):
        r1 = e1.step(acts[t], gov[t])
        r2 = e2.step(acts[t], gov[t])
        # income is reset at period ends only when taxes are on; everything else is identical
        s1, s2 = e1.get_state(), e2.get_state()
        for e in range(4):
            a, b = oracle.parse_state(s1[e]), oracle.parse_state(s2[e])
            assert (a["coin"] == b["coin"]).all() and (a["inv"] == b["inv"]).all()
            assert all((x == y).all() for x, y in zip(a["books"], b["books"]))
        assert (r1[2] == r2[2]).all()


def test_results_do_not_depend_on_batch_placement():
    # T14: draws are keyed by the GLOBAL env id, so env g of a big batch == env 0 of a batch based at g
    cfg = inputs.configs()["tiny_dense"]
    acts, gov = inputs.action_stream(cfg, 30, E=6)
    big = make(6, cfg["N"], cfg["R"], cfg["params"], seed=5)
    one = make(1, cfg["N"], cfg["R"], dict(cfg["params"], env_id_base=4), seed=5)
    for t in range(30):
        ob, og, rb, _ = big.step(acts[t], gov[t])
        o1, g1, r1, _ = one.step(acts[t, 4:5], gov[t, 4:5])
        assert (ob[4] == o1[0]).all() and (og[4] == g1[0]).all() and (rb[4] == r1[0]).all()
    assert (big.get_state(4, 1) == one.get_state()).all()
    # stepping a sub-range leaves the other envs untouched
    before = big.get_state(0, 1).copy()
    big.step(acts[0, 2:4], gov[0, 2:4], env_begin=2)
    assert (big.get_state(0, 1) == before).all()


def test_book_cap_by_arrival_order():
    # G15: the j-th candidate in arrival order on a book is accepted iff n_rest + j < K
    cfg = inputs.configs()["tiny_dense"]
    p = dict(cfg["params"], book_cap=2, starting_coin=50.0)
    a = Act(2, 10)
    env = make(1, 4, 2, p, seed=1)
    env.step([[a.buy(0, 0)] * 4], gov0(env))
    s = st(env)
    assert len(s["books"][0]) == 2 and s["counters"][1] == 2 and s["counters"][2] == 2
    placed = sorted(s["books"][0][:, 1].tolist())
    # the accepted two are the first two in (key, agent) order: recompute the keys from Philox
    L = oracle.lib()
    import ctypes as C
    keys = []
    for i in range(4):
        c, k, o = (C.c_uint32 * 4)(0, i, 0, 0), (C.c_uint32 * 2)(1, 0), (C.c_uint32 * 4)()
        L.orc_philox4x32_10(c, k, o)
        keys.append((o[2], i))
    assert placed == sorted(i for _, i in sorted(keys)[:2])
    # next step: book already holds 2 -> everything rejected
    env.step([[a.buy(0, 0)] * 4], gov0(env))
    assert st(env)["counters"][1] == 2


def test_env_wide_tail_of_the_population_rows_is_identical_for_all_agents():
    """f2 rests on this (market statistics are global; rates and timers are per env): columns
    3R + 4 .. of the population observation do not depend on the agent."""
    cfg = inputs.configs()["tiny_dense"]
    E, N, R = 4, cfg["N"], cfg["R"]
    o = oracle.OracleEnv(E, N, R, cfg["params"])
    o.reset(2)
    acts, gov = inputs.action_stream(cfg, 40, seed=2, E=E)
    varied = 0
    for t in range(40):
        pop, _, _, _ = o.step(acts[t], gov[t])
        tail = pop[:, :, 3 * R + 4:]
        assert (tail == tail[:, :1, :]).all()
        varied += int((pop[:, :, :3 * R + 4] != pop[:, :1, :3 * R + 4]).any())
    assert varied > 0  # while the private block does differ between agents


@pytest.mark.parametrize("name,E,steps", [("config2_paper", 5, 60), ("tiny_dense", 8, 50), ("section5_r4", 3, 40)])
def test_dump_invariant_checker_accepts_the_oracle_and_rejects_a_broken_dump(name, E, steps):
    # parity.check_dump_invariants is what the GPU tests run on every env of the full-size launches
    from parity import check_dump_invariants
    cfg = inputs.configs()[name]
    o = oracle.OracleEnv(E, cfg["N"], cfg["R"], cfg["params"])
    o.reset(2)
    cdf = inputs.action_cdf(cfg)
    for _ in range(steps):
        a, g = o.draw_actions(cdf)
        o.step(a, g, want_obs=False)
    w = np.asarray(o.get_state())
    check_dump_invariants(w, cfg, steps)
    B = len(cfg["params"]["thresholds"]) + 1
    bad = w.copy()
    bad[0, 13 + B + cfg["R"] + 1] += 1          # agent 0's escrowed coin no longer equals its live bids
    with pytest.raises(AssertionError):
        check_dump_invariants(bad, cfg, steps)


def test_sharded_oracle_helper_equals_one_oracle():
    """tests/parity.py's OracleShards (many copies of the oracle on host threads, used by the full-size GPU parity
    tests) returns exactly what one oracle over the same global env ids returns."""
    import sys, os
    sys.path.insert(0, os.path.dirname(__file__))
    from parity import OracleShards

    cfg = inputs.configs()["config2_paper"]
    params = dict(cfg["params"], env_id_base=5)
    cdf = inputs.action_cdf(cfg)
    runs = [(0, 5), (9, 3)]
    sh = OracleShards(cfg["N"], cfg["R"], params, 11, runs, threads=3, per_shard=2)
    ones = [make(n, cfg["N"], cfg["R"], dict(params, env_id_base=5 + lo), seed=11) for lo, n in runs]
    assert sh.n == 8 and sh.ids.tolist() == [0, 1, 2, 3, 4, 9, 10, 11]
    outs = sh.advance(12, cdf=cdf, keep=[3, 11])
    for s in range(12):
        for k, o in enumerate(ones):
            a, g = o.draw_actions(cdf)
            res = o.step(a, g, want_obs=s in (3, 11))
            if s in (3, 11):
                lo = 0 if k == 0 else 5
                for j, ref in enumerate((a, g) + tuple(res)):
                    assert np.array_equal(outs[s][j][lo:lo + o.E], ref), (s, k, j)
    assert np.array_equal(sh.state(), np.concatenate([o.get_state() for o in ones]))
    # supplied actions, every step kept
    acts, gov = inputs.action_stream(cfg, 4, seed=2, E=8)
    outs = sh.advance(4, actions=acts, gov_actions=gov, keep=range(4))
    for s in range(4):
        for k, o in enumerate(ones):
            lo = 0 if k == 0 else 5
            res = o.step(acts[s][lo:lo + o.E], gov[s][lo:lo + o.E])
            assert np.array_equal(outs[s][4][lo:lo + o.E], res[2])
    assert np.array_equal(sh.state(), np.concatenate([o.get_state() for o in ones]))


# ---------------- f4: episodes and auto-reset (G44) ----------------
def test_episode_keying_and_begin_episode(small_params):
    """Every random draw of an episode is keyed by (seed, env, agent, t, stream | episode << 8): episode 0 draws what
    G30's counters draw (all other tests pin that), a later episode is recomputed here from orc_philox4x32_10."""
    import ctypes as C

    L = oracle.lib()

    def philox(ctr, key):
        c, k, o = (C.c_uint32 * 4)(*ctr), (C.c_uint32 * 2)(*key), (C.c_uint32 * 4)()
        L.orc_philox4x32_10(c, k, o)
        return list(o)

    p = dict(small_params, starting_coin=15.0, env_id_base=9)          # uniform skills: skill = (x >> 8) * 2^-24
    seed = 0xABCDEF0123
    key = [seed & 0xFFFFFFFF, seed >> 32]
    env = make(2, 3, 2, p, seed=seed)
    first = env.get_state().copy()
    assert [st(env, e)["episode"] for e in range(2)] == [0, 0]
    acts, gov = inputs.action_stream(dict(E=2, N=3, R=2, T=50, seed=1, action_mix="uniform", params=p), 5, seed=1, E=2)
    for t in range(5):
        env.step(acts[t], gov[t], want_obs=False)
    env.begin_episode(3, env_begin=1, env_count=1)                      # env 1 only
    s0, s1 = st(env, 0), st(env, 1)
    assert s0["t"] == 5 and s0["episode"] == 0 and s1["t"] == 0 and s1["episode"] == 3
    assert (s1["coin"] == 15.0).all() and not s1["inv"].any() and (s1["labor"] == 0).all() and all(len(b) == 0 for b in s1["books"])
    assert s1["counters"].sum() >= 0 and (s1["counters"] == oracle.parse_state(env.get_state()[1])["counters"]).all()
    for i in range(3):
        x = philox([9 + 1, i, 0, 16 | (3 << 8)], key)                  # skill draws d = 0, 1, 2 are words 0, 1, 2 of block 0
        want = [np.float32((w >> 8) * 2.0 ** -24) for w in x[:3]]
        assert s1["SG"][i].tolist() == want[:2] and s1["SC"][i] == want[2]
    assert (s1["SG"] != oracle.parse_state(first[1])["SG"]).any()        # not the skills of episode 0
    # the step draws of the new episode: the arrival key of a placed order is word 2 of stream 0 | 3 << 8
    cdf = inputs.action_cdf(dict(E=2, N=3, R=2, T=50, seed=1, action_mix="uniform", params=p))
    a1, _ = env.draw_actions(cdf, env_begin=1, env_count=1)
    x0 = philox([10, 0, 0, 0 | (3 << 8)], key)[0]
    assert a1[0, 0] == int(np.searchsorted(cdf.astype(np.uint64), x0, side="right"))
    env.begin_episode(0, env_begin=1, env_count=1)
    assert (env.get_state()[1][:6] == first[1][:6]).all() and (st(env, 1)["SG"] == oracle.parse_state(first[1])["SG"]).all()


def test_auto_reset_equals_reset_T_steps_reset_T_steps():
    """orc_step_auto over 2 T + 3 steps = episode 0 for T steps, begin_episode(1), T steps, begin_episode(2), 3 steps; the
    observation of the step that ends an episode is the one of the fresh state; rewards and done are the step's own."""
    cfg = inputs.configs()["tiny_dense"]
    T, E = cfg["T"], 3
    acts, gov = inputs.action_stream(cfg, 2 * T + 3, seed=5, E=E)
    a = make(E, cfg["N"], cfg["R"], cfg["params"], seed=5)
    b = make(E, cfg["N"], cfg["R"], cfg["params"], seed=5)
    n_done = 0
    for t in range(2 * T + 3):
        pa, ga, ra, da = a.step(acts[t], gov[t], auto_reset=True)
        pb, gb, rb, db = b.step(acts[t], gov[t])
        assert np.array_equal(ra, rb) and np.array_equal(da, db)
        if (t + 1) % T == 0:
            assert (da == 1).all()
            n_done += 1
            b.begin_episode((t + 1) // T)
            pb, gb = b.observe()
            assert pb[0, 0, -1] == 0.0 and pb[0, 0, 0] == np.float32(cfg["params"]["starting_coin"]) * np.float32(0.01)
        else:
            assert (da == 0).all()
        assert np.array_equal(pa, pb) and np.array_equal(ga, gb)
        assert np.array_equal(a.get_state(), b.get_state())
    assert n_done == 2 and st(a)["episode"] == 2 and st(a)["t"] == 3
    # the second episode is not a replay of the first
    c = make(E, cfg["N"], cfg["R"], cfg["params"], seed=5)
    for t in range(3):
        c.step(acts[2 * T + t], gov[2 * T + t], want_obs=False)
    assert (st(c)["inv"] != st(a)["inv"]).any() or (st(c)["SG"] != st(a)["SG"]).any()
