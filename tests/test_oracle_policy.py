"""Pins of the a12 oracle (oracle/policy.py): bf16 rounding, the MLP forward, softmax sampling.
None of these retype the oracle's own formula: they use hand-computed values, torch's bfloat16
cast and torch.nn.functional.linear as independent references, and closed-form special cases."""
import numpy as np
import pytest
import torch

from oracle import policy as P
from paper_2410_22165_b200 import inputs


def test_bf16_round_hand_values():
    # 8 significant bits, ties to even: 1 + 2^-8 is a tie between 1 and 1 + 2^-7 -> even mantissa (1.0);
    # 1 + 3 * 2^-8 is a tie between 1 + 2^-7 and 1 + 2^-6 -> 1 + 2^-6
    assert P.bf16_round(1.0) == 1.0
    assert P.bf16_round(1.0 + 2.0 ** -8) == 1.0
    assert P.bf16_round(1.0 + 3 * 2.0 ** -8) == 1.0 + 2.0 ** -6
    assert P.bf16_round(1.0 + 2.0 ** -8 + 2.0 ** -20) == 1.0 + 2.0 ** -7
    assert P.bf16_round(-0.3) == -0.30078125          # 0.3 = 1.2 * 2^-2; 1.2 -> 154/128
    assert P.bf16_round(0.0) == 0.0
    # tanh(0.5) = 0.46211716 = 1.84846864 * 2^-2 -> 237/128 * 2^-2
    assert P.bf16_round(np.tanh(0.5)) == 237.0 / 512.0


def test_bf16_round_matches_torch_cast():
    rng = np.random.default_rng(0)
    x = np.concatenate([rng.standard_normal(20000), rng.standard_normal(2000) * 1e-3, rng.standard_normal(2000) * 300]).astype(np.float32)
    want = torch.from_numpy(x).to(torch.bfloat16).to(torch.float64).numpy()
    got = P.bf16_round(x.astype(np.float64))
    assert np.array_equal(got, want)


def test_bf16_bits_roundtrip_with_input_generator():
    x = np.array([1.0, -2.5, 0.02, 3.14159], np.float32)
    bits = inputs._to_bf16_bits(x)
    assert np.array_equal(P.bf16_bits_to_f64(bits), torch.from_numpy(x).to(torch.bfloat16).to(torch.float64).numpy())


def _net(w1, w2, w3, b1, b2, b3):
    f = lambda a: inputs._to_bf16_bits(np.asarray(a, np.float32))
    return dict(w1=f(w1), w2=f(w2), w3=f(w3), b1=np.asarray(b1, np.float32), b2=np.asarray(b2, np.float32),
                b3=np.asarray(b3, np.float32))


def test_hand_computed_network():
    # 1 -> 2 -> 2 -> 2, every weight exactly representable in bf16
    net = _net([[0.5], [-0.5]], [[1.0, 0.0], [0.0, 2.0]], [[1.0, 1.0], [1.0, -1.0]], [0, 0], [0, 0], [0.25, 0])
    # x = 1: h1 = bf16(tanh(+-0.5)) = +-237/512
    h1 = 237.0 / 512.0
    # h2 = bf16(tanh(h1)), bf16(tanh(-2 h1)): computed by hand from math.tanh and 8-bit rounding
    import math
    def r8(v):
        m, e = math.frexp(v)
        return math.ldexp(round(m * 256), e - 8)
    h2a, h2b = r8(math.tanh(h1)), r8(math.tanh(-2 * h1))
    want = np.array([[h2a + h2b + 0.25, h2a - h2b]])
    got = P.mlp_logits(net, np.array([[1.0]], np.float32))
    assert np.allclose(got, want, rtol=0, atol=1e-15)


@pytest.mark.parametrize("bias_std", [0.0, 0.05])
def test_forward_against_torch_linear(bias_std):
    cfg = inputs.configs()["config5_policy"]
    pop, gov = inputs.policy_weights(cfg, seed=3, bias_std=bias_std)
    rng = np.random.default_rng(1)
    for net, d_in in ((pop, pop["w1"].shape[1]), (gov, gov["w1"].shape[1])):
        x = (rng.standard_normal((50, d_in)) * 0.7).astype(np.float32)
        tw = lambda k: torch.from_numpy(net[k].astype(np.int32) << 16).view(torch.float32).to(torch.float64)
        tb = lambda k: torch.from_numpy(net[k]).to(torch.float64)
        h = torch.from_numpy(x).to(torch.bfloat16).to(torch.float64)
        h = torch.tanh(torch.nn.functional.linear(h, tw("w1"), tb("b1"))).to(torch.bfloat16).to(torch.float64)
        h = torch.tanh(torch.nn.functional.linear(h, tw("w2"), tb("b2"))).to(torch.bfloat16).to(torch.float64)
        want = torch.nn.functional.linear(h, tw("w3"), tb("b3")).numpy()
        got = P.mlp_logits(net, x)
        assert got.shape == want.shape
        assert np.allclose(got, want, rtol=1e-12, atol=1e-14)


def test_weight_statistics_of_the_generator():
    cfg = inputs.configs()["config5_policy"]
    pop, gov = inputs.policy_weights(cfg, seed=0)
    d = inputs.policy_dims(cfg)
    assert pop["w1"].shape == (128, d["D_pop"]) == (128, 37) and pop["w3"].shape == (d["A"], 128) == (65, 128)
    assert gov["w1"].shape == (128, d["D_gov"]) == (128, 27) and gov["w3"].shape == (147, 128)
    w = P.bf16_bits_to_f64(pop["w2"])
    assert abs(w.mean()) < 1e-3 and abs(w.std() - 0.02) < 1e-3     # N(0, 0.02), BASELINE.json configs[4]
    assert not pop["b1"].any() and not gov["b3"].any()


def test_sampling_special_cases():
    A = 65
    for u in (0.0, 0.3, 0.5, 0.999999):
        assert P.sample(np.zeros(A), u) == int(u * A)               # uniform logits: floor(u A)
    l = np.full(7, -50.0); l[4] = 50.0
    assert P.sample(l, 1e-9) == 4 and P.sample(l, 0.99) == 4         # one dominant logit (p_other = e^-100)
    c = P.softmax_cdf([0.0, np.log(3.0)])                           # p = (1/4, 3/4)
    assert np.allclose(c, [0.25, 1.0])
    assert P.sample([0.0, np.log(3.0)], 0.2499) == 0 and P.sample([0.0, np.log(3.0)], 0.25) == 1
    # shift invariance of softmax
    rng = np.random.default_rng(5)
    l = rng.standard_normal(21)
    assert np.allclose(P.softmax_cdf(l), P.softmax_cdf(l + 123.0))


def test_sample_consistent_brute_force():
    rng = np.random.default_rng(9)
    for _ in range(200):
        l = rng.standard_normal(11)
        u = float(rng.random())
        a = P.sample(l, u)
        p = np.exp(l) / np.exp(l).sum()
        assert p[:a].sum() <= u + 1e-12 and u < p[:a + 1].sum() + 1e-12   # brute-force interval membership
        assert P.sample_consistent(l, u, a, 0.0)
        others = [b for b in range(11) if b != a and not P.sample_consistent(l, u, b, 1e-3)]
        assert len(others) >= 8                                        # only near neighbours can be eps-consistent


def test_philox_u_uses_the_pinned_generator():
    # T11 known answer: counter = key = 0 -> 6627e8d5 e169c58d bc57ac4c 9b00dbd8
    assert P.philox_u(0, 0, 0, 0, 0, 0) == (0x6627e8d5 >> 8) / 16777216.0
    assert P.philox_u(0, 0, 0, 0, 0, 3) == (0x9b00dbd8 >> 8) / 16777216.0


# ---- f1: masked categorical ----

def test_masked_softmax_hand_values_and_library():
    from scipy.special import softmax
    l = np.array([0.0, 5.0, 0.0, -1.0, 0.0])
    m = np.array([1, 0, 1, 0, 1])
    c = P.softmax_cdf(l, m)
    assert np.allclose(c, [1 / 3, 1 / 3, 2 / 3, 2 / 3, 1.0], atol=1e-15)      # the dominant logit is unavailable
    assert P.sample(l, 0.33, m) == 0 and P.sample(l, 0.34, m) == 2 and P.sample(l, 0.999, m) == 4
    rng = np.random.default_rng(0)
    for _ in range(50):
        l = rng.normal(0, 2, 17)
        m = rng.random(17) < 0.5
        m[rng.integers(17)] = True
        c = P.softmax_cdf(l, m)
        p = np.diff(np.concatenate([[0.0], c]))
        assert np.all(p[~m] == 0.0)
        idx = np.flatnonzero(m)
        assert np.allclose(p[idx][:-1], softmax(l[idx])[:-1], atol=1e-12)     # = softmax over the available sub-vector
        for u in rng.random(20):
            a = P.sample(l, float(u), m)
            assert m[a] and P.sample_consistent(l, float(u), a, 0.0, m)


def test_mask_of_ones_changes_nothing():
    rng = np.random.default_rng(1)
    l = rng.normal(0, 1, 44)
    assert np.array_equal(P.softmax_cdf(l), P.softmax_cdf(l, np.ones(44, np.uint8)))
    for u in rng.random(30):
        assert P.sample(l, float(u)) == P.sample(l, float(u), np.ones(44, np.uint8))
