"""Pins of the f1 oracle (orc_action_mask): hand-checked states, and mask soundness / completeness
against the step rules: with no book cap an action is available exactly when submitting
it does not bump the env's invalid-action counter.  The step's validity tests are separate code
from the mask function, so a wrong precondition in either shows up."""
import numpy as np
import pytest

import oracle
from conftest import Act
from paper_2410_22165_b200 import inputs


def test_mask_hand_examples(small_params):
    p = dict(small_params, starting_coin=0.0)
    o = oracle.OracleEnv(1, 3, 2, p)
    o.reset(0)
    act = Act(2, 10)
    # agent 0: coin 4.5, inv (0, 3): buys up to price 4, sells r1 only, no craft (needs 2 of BOTH resources)
    o.set_agent(0, 0, 4.5, [0, 3], [1.0, 1.0], 1.0)
    # agent 1: coin 0, inv (2, 2): craft available, no buys, both sells
    o.set_agent(0, 1, 0.0, [2, 2], [1.0, 1.0], 1.0)
    # agent 2: coin 100, nothing else
    o.set_agent(0, 2, 100.0, [0, 0], [1.0, 1.0], 1.0)
    m = o.action_mask()[0]
    assert m.shape == (3, act.A) and m.dtype == np.uint8
    for i in range(3):
        assert m[i, act.gather(0)] == 1 and m[i, act.gather(1)] == 1 and m[i, act.noop] == 1
    assert m[0, act.craft()] == 0 and m[1, act.craft()] == 1 and m[2, act.craft()] == 0
    assert [int(m[0, act.buy(0, k)]) for k in range(10)] == [1, 1, 1, 1, 0, 0, 0, 0, 0, 0]       # prices 1..10, coin 4.5
    assert [int(m[0, act.buy(1, k)]) for k in range(10)] == [1, 1, 1, 1, 0, 0, 0, 0, 0, 0]
    assert m[0, act.sell(0, 0):act.sell(0, 9) + 1].sum() == 0 and m[0, act.sell(1, 0):act.sell(1, 9) + 1].sum() == 10
    assert m[1, act.buy(0, 0):act.buy(1, 9) + 1].sum() == 0 and m[1, act.sell(0, 0):act.sell(1, 9) + 1].sum() == 20
    assert m[2, act.buy(0, 0):act.buy(1, 9) + 1].sum() == 20 and m[2, act.sell(0, 0):act.sell(1, 9) + 1].sum() == 0


def test_mask_order_cap(small_params):
    p = dict(small_params, max_active_orders=2, order_expiry=40)
    o = oracle.OracleEnv(1, 2, 2, p)
    o.reset(0)
    act = Act(2, 10)
    gov = np.zeros((1, 3), np.int32)
    o.set_agent(0, 0, 50.0, [5, 5], [1.0, 1.0], 1.0)
    o.step(np.array([[act.buy(0, 0), act.noop]], np.int32), gov)      # bids that cannot match (no asks)
    m = o.action_mask()[0]
    assert m[0, act.buy(0, 0)] == 1 and m[0, act.sell(1, 9)] == 1
    o.step(np.array([[act.buy(1, 0), act.noop]], np.int32), gov)
    m = o.action_mask()[0]                                            # two live orders = the cap
    assert m[0, act.buy(0, 0):act.sell(1, 9) + 1].sum() == 0
    assert m[0, act.gather(0)] == 1 and m[0, act.craft()] == 1 and m[0, act.noop] == 1


@pytest.mark.parametrize("name,craft_mode", [("tiny_dense", 0), ("tiny_dense", 1), ("config2_paper", 0)])
def test_mask_is_sound_and_complete_against_the_step(name, craft_mode):
    cfg = inputs.configs()[name]
    params = dict(cfg["params"], craft_mode=craft_mode, max_active_orders=3, episode_length=1000)
    E, N, R = 2, cfg["N"], cfg["R"]
    o = oracle.OracleEnv(E, N, R, params)
    o.reset(5)
    acts, gov = inputs.action_stream(dict(cfg, params=params), 60, seed=5, E=E)
    A = o.A
    rng = np.random.default_rng(2)
    checked = 0
    for t in range(60):
        o.step(acts[t] % A, gov[t], want_obs=False)
        if t % 4:
            continue
        m = o.action_mask()
        # probe: a replayed copy of the batch (the oracle is deterministic) in which agent i of env e submits
        # action a and everyone else a no-op
        for _ in range(12):
            e, i, a = int(rng.integers(E)), int(rng.integers(N)), int(rng.integers(A))
            probe = oracle.OracleEnv(E, N, R, params)
            probe.reset(5)
            for u in range(t + 1):
                probe.step(acts[u] % A, gov[u], want_obs=False)
            before = oracle.parse_state(probe.get_state()[e])["counters"][2]
            a_all = np.full((E, N), A - 1, np.int32)
            a_all[e, i] = a
            probe.step(a_all, gov[t], want_obs=False)
            after = oracle.parse_state(probe.get_state()[e])["counters"][2]
            assert (after == before) == bool(m[e, i, a]), "t=%d env %d agent %d action %d: mask %d, invalid counter %d -> %d" % (t, e, i, a, m[e, i, a], before, after)
            checked += 1
    assert checked >= 150
