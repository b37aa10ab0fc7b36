"""Pins of the oracle's rule-level functions against what the paper and the mathematics fix
(SURVEY.md 8(c) T1-T13).  CPU only.  A dropped term, wrong sign/index or transposed operand
in oracle/econojax_oracle.c must fail at least one test here or in test_oracle_env.py."""
import ctypes as C
import decimal
import os

import numpy as np
import pytest

import oracle

L = oracle.lib()
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    for line in open(os.path.join(GOLD, name)):
        line = line.strip()
        if line and not line.startswith("#"):
            yield line


def _f32(vals):
    return (C.c_float * len(vals))(*vals)


def philox(ctr, key):
    c, k, o = (C.c_uint32 * 4)(*ctr), (C.c_uint32 * 2)(*key), (C.c_uint32 * 4)()
    L.orc_philox4x32_10(c, k, o)
    return list(o)


# ---- T11 RNG ----
def test_philox_known_answers():
    n = 0
    for line in _rows("philox4x32_10_kat.txt"):
        w = [int(x, 16) for x in line.split()]
        assert philox(w[0:4], w[4:6]) == w[6:10]
        n += 1
    assert n == 3


def test_philox_counter_and_key_sensitivity():
    base = philox([1, 2, 3, 4], [5, 6])
    for pos in range(4):
        c = [1, 2, 3, 4]
        c[pos] ^= 1
        assert philox(c, [5, 6]) != base
    assert philox([1, 2, 3, 4], [5, 7]) != base and philox([1, 2, 3, 4], [4, 6]) != base


def test_u01_is_top_24_bits():
    assert L.orc_u01(0) == 0.0
    assert L.orc_u01(0xFF) == 0.0
    assert L.orc_u01(0x100) == 2.0 ** -24
    assert L.orc_u01(0xFFFFFFFF) == 1.0 - 2.0 ** -24
    assert L.orc_u01(0x80000000) == 0.5


# ---- golden worked examples (T1, T2, T3, T4) ----
def _kv(s):
    return dict(item.split("=") for item in s.split())


def test_paper_worked_examples():
    seen = set()
    for line in _rows("paper_worked_examples.txt"):
        kind, inp, exp, _cite = [x.strip() for x in line.split("|")]
        kv = _kv(inp)
        seen.add(kind)
        if kind == "tax":
            thr = [float(x) for x in kv["thresholds"].split(",")]
            rates = [float(x) for x in kv["rates"].split(",")]
            got = L.orc_marginal_tax(float(kv["income"]), _f32(thr), _f32(rates), len(rates))
            assert got == float(exp)  # exactly 35.0f / 4.0f in binary32 with mul-then-add
        elif kind == "actions":
            assert L.orc_num_actions(int(kv["R"]), int(kv["P"]), oracle.CRAFT_SINGLE, int(kv["noop"])) == int(exp)
        elif kind == "gather":
            u = np.float32(float(kv["rho"]) / 1.1)
            # choose u so that fl(u*1.1f) is within an ulp of rho; the cases are far from an integer boundary
            assert L.orc_gather_amount(float(kv["SG"]), float(u)) == int(exp)
        elif kind == "utility":
            got = L.orc_utility(float(kv["C"]), float(kv["L"]), float(kv["eta"]))
            assert abs(got - float(exp)) < 1e-12
    assert seen == {"tax", "actions", "gather", "utility"}


def test_action_counts_of_the_five_configs():
    # R + 1 + 2RP + 1; per-resource convert adds R-1 (G3)
    assert L.orc_num_actions(2, 10, 0, 1) == 44
    assert L.orc_num_actions(6, 10, 0, 1) == 128
    assert L.orc_num_actions(3, 10, 0, 1) == 65
    assert L.orc_num_actions(2, 10, 1, 1) == 45
    assert L.orc_num_actions(6, 10, 1, 1) == 133
    assert L.orc_num_actions(2, 5, 0, 0) == 2 + 1 + 20


# ---- T1 tax ----
def test_marginal_tax_properties():
    rng = np.random.default_rng(0)
    thr = [10.0, 20.0, 40.0, 80.0, 160.0, 320.0]
    for _ in range(200):
        rates = [float(np.float32(k / 20)) for k in rng.integers(0, 21, size=7)]
        inc = np.sort(rng.uniform(0, 600, size=20).astype(np.float32))
        taxes = [L.orc_marginal_tax(float(x), _f32(thr), _f32(rates), 7) for x in inc]
        assert all(b >= a - 1e-4 for a, b in zip(taxes, taxes[1:]))  # monotone
        assert all(t <= max(rates) * x * (1 + 1e-6) + 1e-6 for t, x in zip(taxes, inc))
        # independent per-bracket summation in binary64
        edges = [0.0] + thr + [np.inf]
        for x, t in zip(inc, taxes):
            ref = sum(r * max(0.0, min(float(x), hi) - lo) for r, lo, hi in zip(rates, edges[:-1], edges[1:]))
            assert abs(t - ref) <= 1e-5 * max(1.0, ref)
    assert L.orc_marginal_tax(500.0, _f32(thr), _f32([0.0] * 7), 7) == 0.0
    assert L.orc_marginal_tax(500.0, _f32(thr), _f32([1.0] * 7), 7) == 500.0
    # a single bracket is a flat tax
    assert L.orc_marginal_tax(80.0, _f32([0.0]), _f32([0.25]), 1) == 20.0


# ---- T2 utility ----
def test_utility_against_high_precision_evaluation():
    decimal.getcontext().prec = 50
    for Cv, Lv in [(15.0, 0.0), (143.25, 37.05), (0.001, 2.0), (1e4, 0.0)]:
        a = decimal.Decimal(1) - decimal.Decimal(0.27)
        ref = ((decimal.Decimal(Cv).ln() * a).exp() - 1) / a - decimal.Decimal(Lv)
        got = L.orc_utility(Cv, Lv, 0.27)
        assert abs(decimal.Decimal(got) - ref) < decimal.Decimal(1e-11) * max(1, abs(ref))
    assert abs(L.orc_utility(15.0, 0.0, 0.27) - 8.5207625) < 1e-7  # SURVEY T2 (S:294 prints 8.5204, a typo: G35)
    assert L.orc_utility(15.0, 1.0, 0.27) - L.orc_utility(15.0, 0.0, 0.27) == pytest.approx(-1.0, abs=1e-12)


def test_utility_increasing_and_concave_in_coin():
    xs = np.linspace(0.5, 300, 200)
    u = np.array([L.orc_utility(float(x), 0.0, 0.27) for x in xs])
    d1 = np.diff(u)
    assert (d1 > 0).all() and (np.diff(d1) < 0).all()


# ---- T9 gini / welfare ----
def gini(v):
    a = np.asarray(v, np.float32)
    return L.orc_gini(a.ctypes.data_as(C.POINTER(C.c_float)), len(a))


def test_gini_textbook_values():
    assert gini([10, 10, 10]) == 0.0
    assert gini([0, 1]) == 0.5
    assert gini([0, 0, 0]) == 0.0
    assert gini([7]) == 0.0
    assert gini([1, 2, 3, 4]) == pytest.approx(0.25, abs=1e-15)
    # one agent owns everything: (n-1)/n
    assert gini([0, 0, 0, 0, 5]) == pytest.approx(0.8, abs=1e-15)


def test_gini_equals_sorted_rank_form_and_is_invariant():
    rng = np.random.default_rng(1)
    for n in (2, 3, 17, 100):
        for _ in range(20):
            c = rng.gamma(2.0, 50.0, size=n).astype(np.float32)
            g = gini(c)
            s = np.sort(c.astype(np.float64))
            i = np.arange(n)
            ref = ((2 * i - n + 1) * s).sum() / (n * s.sum())  # S:330 equivalent form
            assert g == pytest.approx(ref, abs=1e-12)
            assert gini(rng.permutation(c)) == pytest.approx(g, abs=1e-13)
            assert gini(c * np.float32(4.0)) == pytest.approx(g, abs=1e-13)  # power-of-two scale is exact
            assert 0.0 <= g <= 1.0


def welfare(c, omega):
    a = np.asarray(c, np.float32)
    eq, prod, ug = C.c_double(), C.c_double(), C.c_double()
    L.orc_social_welfare(a.ctypes.data_as(C.POINTER(C.c_float)), len(a), omega, C.byref(eq), C.byref(prod), C.byref(ug))
    return eq.value, prod.value, ug.value


def test_social_welfare_examples():
    assert welfare([10, 10], 1.0) == (1.0, 20.0, 20.0)
    assert welfare([0, 1], 1.0) == (0.5, 1.0, 0.5)
    eq, prod, ug = welfare([3, 9, 1], 0.0)                       # omega = 0 removes the equality weight
    assert (eq, prod, ug) == (1.0, 13.0, 13.0)
    eq, prod, ug = welfare([3, 9, 1], 0.5)
    g = gini([3, 9, 1])
    assert eq == pytest.approx(0.5 * (1 - g) + 0.5) and ug == pytest.approx(eq * 13.0)
    eq, prod, ug = welfare([3, 9, 1], 1.0)                       # Fig.2 "Equality: (1 - gini)"
    assert eq == pytest.approx(1 - g)


# ---- T10 statistics ----
def stats(x):
    a = np.asarray(x, np.float32)
    m, s, med = C.c_double(), C.c_double(), C.c_float()
    L.orc_stats(a.ctypes.data_as(C.POINTER(C.c_float)), len(a), C.byref(m), C.byref(s), C.byref(med))
    return m.value, s.value, med.value


def test_stats_examples_and_numpy_cross_check():
    m, s, med = stats([1, 2, 3])
    assert (m, med) == (2.0, 2.0) and s == pytest.approx(0.816496580927726)
    assert stats([1, 2, 3, 4])[2] == 2.5
    assert stats([4, 1, 3, 2])[2] == 2.5
    rng = np.random.default_rng(2)
    for n in (1, 2, 4, 5, 100, 101, 1000):
        x = rng.gamma(2.0, 30.0, size=n).astype(np.float32)
        x[rng.integers(0, n, size=n // 3)] = x[0]  # ties
        m, s, med = stats(x)
        assert m == pytest.approx(np.mean(x.astype(np.float64)), rel=1e-13)
        assert s == pytest.approx(np.std(x.astype(np.float64)), rel=1e-12, abs=1e-12)
        assert med == np.median(x)  # numpy's float32 midpoint is the same (a+b)*0.5 in binary32


# ---- T5 craft ----
def craft(inv, units, distinct, mode=0, r_named=0):
    a = (C.c_int32 * len(inv))(*inv)
    ok = L.orc_craft_consume(a, len(inv), units, distinct, mode, r_named)
    return ok, list(a)


def test_craft_examples():
    assert craft([3, 2], 2, 2) == (1, [1, 0])
    assert craft([2, 5, 3], 2, 2) == (1, [2, 3, 1])        # consumes from r1 and r2 (most held)
    assert craft([2, 2], 2, 2) == (1, [0, 0])
    assert craft([1, 5], 2, 2) == (0, [1, 5])              # only one resource has enough
    assert craft([2, 2, 2], 2, 2) == (1, [0, 0, 2])        # ties -> lowest index (G7)
    assert craft([4, 4, 9, 4, 1], 2, 3) == (1, [2, 2, 7, 4, 1])  # P:156 "2 of each of 3 resources" out of 5
    assert craft([9, 1, 1, 1, 1], 2, 3) == (0, [9, 1, 1, 1, 1])
    assert craft([0, 3], 2, 2, mode=1, r_named=1) == (1, [0, 1])  # PER_RESOURCE variant (G3)
    assert craft([0, 1], 2, 2, mode=1, r_named=1) == (0, [0, 1])


# ---- T4 gather boundaries ----
def test_gather_amount_boundaries():
    one_minus = float(np.nextafter(np.float32(1.0), np.float32(0.0)))
    assert L.orc_gather_amount(0.0, one_minus) == 1   # rho can exceed 1 (up to 1.1)
    assert L.orc_gather_amount(0.0, 0.9) == 0         # 0.99 < 1
    assert L.orc_gather_amount(0.0, 0.0) == 0
    assert L.orc_gather_amount(3.0, 0.0) == 3
    assert L.orc_gather_amount(9.95, one_minus) == 11


# ---- T6 matching ----
def run_match(bids, asks):
    """bids/asks: lists of (price, owner, placed_at, key). Returns (trades, remaining bids, remaining asks)."""
    nb, na = C.c_int32(len(bids)), C.c_int32(len(asks))
    B = (oracle.OrcOrder * max(1, len(bids)))(*[oracle.OrcOrder(*o) for o in bids])
    A = (oracle.OrcOrder * max(1, len(asks)))(*[oracle.OrcOrder(*o) for o in asks])
    T = (oracle.OrcTrade * 64)()
    n = L.orc_match_book(B, C.byref(nb), A, C.byref(na), T, 64)
    trades = [(T[i].buyer, T[i].seller, T[i].bid_price, T[i].ask_price, T[i].price) for i in range(n)]
    rb = [(B[i].price, B[i].owner, B[i].placed_at, B[i].key) for i in range(nb.value)]
    ra = [(A[i].price, A[i].owner, A[i].placed_at, A[i].key) for i in range(na.value)]
    return trades, rb, ra


def test_matching_worked_examples():
    # ask@4 placed t=1, bid@6 placed t=2 -> trade at 6, the price of the order placed last
    assert run_match([(6, 0, 2, 0)], [(4, 1, 1, 0)])[0] == [(0, 1, 6, 4, 6)]
    # the resting bid was first, the ask arrives last -> trade at the ask's price
    assert run_match([(6, 0, 1, 0)], [(4, 1, 2, 0)])[0] == [(0, 1, 6, 4, 4)]
    # bid < ask: no trade
    tr, rb, ra = run_match([(4, 0, 1, 0)], [(6, 1, 1, 0)])
    assert tr == [] and len(rb) == 1 and len(ra) == 1
    # bids 8 (t1), 6 (t2); ask 5 (t3): the high bid is evaluated first, price 5, refund 3
    tr, rb, ra = run_match([(8, 0, 1, 0), (6, 1, 2, 0)], [(5, 2, 3, 0)])
    assert tr == [(0, 2, 8, 5, 5)] and rb == [(6, 1, 2, 0)] and ra == []
    # equal prices: the older order goes first
    tr, rb, _ = run_match([(6, 0, 5, 9), (6, 1, 3, 9)], [(6, 2, 7, 0)])
    assert tr == [(1, 2, 6, 6, 6)] and rb == [(6, 0, 5, 9)]
    # same price and step: the tie key decides, then the agent index (G11)
    tr, _, _ = run_match([(6, 0, 5, 9), (6, 1, 5, 3)], [(6, 2, 7, 0)])
    assert tr[0][0] == 1
    tr, _, _ = run_match([(6, 4, 5, 3), (6, 1, 5, 3)], [(6, 2, 7, 0)])
    assert tr[0][0] == 1
    # both placed in the same step: the larger tie key is "placed last"
    assert run_match([(7, 0, 5, 10)], [(3, 1, 5, 20)])[0] == [(0, 1, 7, 3, 3)]
    assert run_match([(7, 0, 5, 30)], [(3, 1, 5, 20)])[0] == [(0, 1, 7, 3, 7)]
    # an agent's own bid and ask trade like any other pair (G12)
    assert run_match([(5, 3, 1, 0)], [(5, 3, 2, 0)])[0] == [(3, 3, 5, 5, 5)]


def _arrival(o):
    return (o[2], o[3], o[1])


def _sort_and_zip(bids, asks):
    """Independent formulation: rank both sides, pair rank i with rank i while bid >= ask."""
    sb = sorted(bids, key=lambda o: (-o[0],) + _arrival(o))
    sa = sorted(asks, key=lambda o: (o[0],) + _arrival(o))
    trades = []
    for b, a in zip(sb, sa):
        if b[0] < a[0]:
            break
        price = b[0] if _arrival(b) > _arrival(a) else a[0]
        trades.append((b[1], a[1], b[0], a[0], price))
    return trades


def test_matching_brute_force_on_tiny_books():
    rng = np.random.default_rng(3)
    for case in range(1500):
        nb, na = rng.integers(0, 11, size=2)
        mk = lambda n: [(int(rng.integers(1, 7)), int(rng.integers(0, 6)), int(rng.integers(0, 4)),
                         int(rng.integers(0, 3))) for _ in range(n)]
        bids, asks = mk(nb), mk(na)
        # no two orders of one owner in one step on the same side (one action per agent per step)
        uniq = lambda os: list({(o[1], o[2]): o for o in os}.values())
        bids, asks = uniq(bids), uniq(asks)
        asks = [a for a in asks if (a[1], a[2]) not in {(b[1], b[2]) for b in bids}]
        trades, rb, ra = run_match(bids, asks)
        assert trades == _sort_and_zip(bids, asks)
        # histogram count q = max_p min(#bids >= p, #asks <= p)
        q = max([min(sum(b[0] >= p for b in bids), sum(a[0] <= p for a in asks)) for p in range(1, 8)] + [0])
        assert len(trades) == q
        for (_, _, bp, ap, pr) in trades:
            assert ap <= pr <= bp and pr in (ap, bp)
        if rb and ra:
            assert max(b[0] for b in rb) < min(a[0] for a in ra)  # uncrossed afterwards
        assert len(rb) == len(bids) - q and len(ra) == len(asks) - q
        assert sorted(rb + [b for b in bids if b not in rb]) == sorted(bids)


# ---- f3: skill growth (G41) ----

def _progress(skill, rate=0.005, mx=5.0):
    import ctypes as C
    L = oracle.lib()
    L.orc_progress_skill.restype = C.c_float
    L.orc_progress_skill.argtypes = [C.c_float, C.c_float, C.c_float]
    return float(L.orc_progress_skill(skill, rate, mx))


def test_skill_growth_closed_form_and_limits():
    # 0.5 % at skill << max, shrinking linearly to 0 at the maximum skill level of 5
    assert abs(_progress(1.0) - 1.004) < 1e-6            # 1 + 1 * 0.005 * (1 - 1/5), also S:104
    assert _progress(5.0) == 5.0 and _progress(0.0) == 0.0
    assert abs(_progress(2.5) - (2.5 + 2.5 * 0.005 * 0.5)) < 1e-6
    assert abs(_progress(1e-3) / 1e-3 - 1.005) < 1e-5    # the full 0.5 % far from the cap
    xs = np.linspace(0.0, 5.0, 2001, dtype=np.float32)
    ys = np.array([_progress(float(x)) for x in xs])
    assert np.all(ys >= xs) and np.all(ys <= 5.0)        # never decreases, never passes the cap
    gain = ys[1:-1] / xs[1:-1] - 1.0
    assert np.all(np.diff(gain) <= 1e-6)                  # "this bonus shrinks as the agent approaches the maximum"
    assert _progress(1.0, rate=0.0) == 1.0


def test_skill_growth_in_the_step(small_params):
    from conftest import Act
    act = Act(2, 10)
    gov = np.zeros((1, 3), np.int32)
    for rate in (0.0, 0.005):
        p = dict(small_params, skill_growth_rate=rate, skill_max=5.0)
        o = oracle.OracleEnv(1, 3, 2, p)
        o.reset(0)
        o.set_agent(0, 0, 0.0, [0, 0], [1.0, 2.0], 3.0)
        o.set_agent(0, 1, 0.0, [2, 2], [1.0, 2.0], 3.0)
        o.set_agent(0, 2, 0.0, [0, 0], [1.0, 2.0], 3.0)
        o.step(np.array([[act.gather(1), act.craft(), act.craft()]], np.int32), gov)   # agent 2's craft is invalid
        s = oracle.parse_state(o.get_state()[0])
        g = lambda x: _progress(x) if rate else x
        assert s["SG"][0].tolist() == [1.0, np.float32(g(2.0))]      # only the gathered resource's skill grows
        assert s["SC"][0] == 3.0 and s["SG"][1].tolist() == [1.0, 2.0]
        assert s["SC"][1] == np.float32(g(3.0))                       # craft: the crafting skill
        assert s["coin"][1] == 30.0                                   # payout used the skill BEFORE the increase
        assert s["SC"][2] == 3.0                                      # an invalid craft teaches nothing


# ---- f3: normal skill initialisation (G42) ----

def _normal_skill(words, mean=1.0, std=1.0, lo=-1e30, hi=1e30):
    import ctypes as C
    L = oracle.lib()
    L.orc_normal_skill.restype = C.c_float
    L.orc_normal_skill.argtypes = [C.POINTER(C.c_uint32)] + [C.c_float] * 4
    w = (C.c_uint32 * 12)(*[int(x) for x in words])
    return float(L.orc_normal_skill(w, mean, std, lo, hi))


def test_normal_skill_hand_values_and_exact_recomputation():
    from fractions import Fraction
    half = [1 << 31] * 12                       # every uniform 0.5: z = 0, the skill is the mean
    assert _normal_skill(half) == 1.0 and _normal_skill(half, mean=2.5, std=3.0) == 2.5
    assert _normal_skill([0] * 12) == -5.0      # z = -6, the lower end of the support
    assert _normal_skill([0] * 12, lo=0.0, hi=5.0) == 0.0                    # clipped below
    assert _normal_skill([0xFFFFFFFF] * 12, lo=0.0, hi=5.0) == 5.0           # z -> 6: clipped above
    assert _normal_skill([0xFF] * 12) == -5.0   # the low 8 bits of a word are not used (24-bit uniforms, as orc_u01)
    one = [1 << 31] * 11 + [(1 << 31) + (1 << 8)]                            # one lattice step above the mean
    assert _normal_skill(one, mean=0.0) == 2.0 ** -24
    rng = np.random.default_rng(5)
    for _ in range(300):                        # rational arithmetic, one rounding to binary32 at the end
        w = rng.integers(0, 1 << 32, 12, dtype=np.uint64)
        mean, std = np.float32(rng.normal(1, 1)), np.float32(abs(rng.normal(1, 1)))
        z = Fraction(sum(int(x) >> 8 for x in w), 1 << 24) - 6
        exact = Fraction(float(mean)) + Fraction(float(std)) * z
        got = _normal_skill(w, float(mean), float(std))
        assert abs(Fraction(got) - exact) <= abs(exact) * Fraction(1, 1 << 23) + Fraction(1, 1 << 140)
        assert got == float(np.float32(float(exact)))   # float(Fraction) is correctly rounded; the sum fits binary64 here


def test_normal_skill_distribution():
    from scipy import stats
    rng = np.random.default_rng(11)
    w = rng.integers(0, 1 << 32, (40000, 12), dtype=np.uint64)
    z = np.array([_normal_skill(r, mean=0.0, std=1.0) for r in w], np.float64)
    assert abs(z.mean()) < 0.02 and abs(z.std() - 1.0) < 0.02
    assert stats.kstest(z, "norm").statistic < 0.012    # a sample of 40 000 from N(0,1) itself gives ~0.004-0.008
    assert abs(stats.skew(z)) < 0.05 and abs(stats.kurtosis(z) + 0.1) < 0.08   # the twelve-uniform sum has excess kurtosis -0.1


def test_normal_skill_at_reset(small_params):
    p = dict(small_params, skill_init=oracle.SKILL_NORMAL_CLIP, skill_mean=1.0, skill_std=1.0, skill_clip_lo=0.0, skill_clip_hi=5.0)
    o = oracle.OracleEnv(40, 50, 2, p)
    o.reset(3)
    st = [oracle.parse_state(w) for w in o.get_state()]
    sk = np.concatenate([np.concatenate([s["SG"].ravel(), s["SC"].ravel()]) for s in st]).astype(np.float64)
    assert sk.size == 40 * 50 * 3 and sk.min() >= 0.0 and sk.max() <= 5.0
    # N(1,1) clipped at 0: P(skill = 0) = Phi(-1) = 0.1587; mean of max(0, X) = Phi(1) + phi(1) = 1.0833
    assert abs((sk == 0.0).mean() - 0.1587) < 0.015 and abs(sk.mean() - 1.0833) < 0.03
    o2 = oracle.OracleEnv(40, 50, 2, p)
    o2.reset(3)
    assert all((a == b).all() for a, b in zip(o.get_state(), o2.get_state()))          # deterministic
    o2.reset(4)
    assert any((a != b).any() for a, b in zip(o.get_state(), o2.get_state()))          # keyed by the seed
    # draws of different agents / skills / envs are different words (no stream reuse): nearly all values distinct
    assert np.unique(sk[sk > 0]).size > 0.99 * (sk > 0).sum()
