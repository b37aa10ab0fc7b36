"""Seeded synthetic inputs and workload definitions shared by the oracle and the CUDA path.

This module holds NONE of the method's arithmetic: it only names parameter values
(Table 2 of the paper, and BASELINE.json's five configs), and draws the
seeded action streams and action-distribution tables that both sides consume as
inputs.  It imports neither ``oracle`` nor the CUDA binding.

The paper has no dataset: its workloads are agents acting in the simulator
 and trained policies are not available, so the action streams are
seeded random draws shaped as BASELINE.json prescribes.
"""
from __future__ import annotations

import math

import numpy as np

CRAFT_SINGLE, CRAFT_PER_RESOURCE = 0, 1
SKILL_UNIFORM01, SKILL_PARETO_CLIP, SKILL_NORMAL_CLIP = 0, 1, 2


def rate_table(levels: int) -> list:
    """Rate of level k = (float)(k / (levels-1)) (G5); 21 levels of 5% in the paper."""
    return [float(np.float32(k / (levels - 1))) for k in range(levels)]


def default_params() -> dict:
    """Table 2 environment defaults, plus this build's conventions."""
    return dict(
        prices=[2, 4, 6, 8, 10],
        episode_length=1000,
        tax_period=100,
        thresholds=[50.0, 100.0],         # the paper's illustrative [50;100]
        rate_table=rate_table(21),
        allow_noop=1,
        starting_coin=15.0,
        order_expiry=30,
        max_active_orders=15,
        book_cap=0,                       # G15
        craft_units=2,
        craft_distinct=2,
        craft_mode=CRAFT_SINGLE,          # P:156-157, P:350 (G3)
        labor_craft=1.0, labor_gather=1.0, labor_trade=0.05,
        eta=0.27,
        omega=1.0,
        craft_scale=10.0,                 # G6
        taxes_enabled=1,
        skill_init=SKILL_UNIFORM01,
        skill_clip_lo=1.0, skill_clip_hi=10.0,
        obs_scale_coin=0.01, obs_scale_count=0.1, obs_scale_price=0.1, obs_scale_labor=0.01,  # G25
        env_id_base=0,
        skill_growth_rate=0.0,            # f3: 0 = fixed skills; section 5 uses 0.005
        skill_mean=1.0, skill_std=1.0,    # f3: SKILL_NORMAL_CLIP parameters
        skill_max=5.0,
    )


THRESHOLDS_7 = [10.0, 20.0, 40.0, 80.0, 160.0, 320.0]  # G32: synthetic geometric thresholds


def _cfg(E, N, R, T, seed, action_mix="uniform", **over):
    p = default_params()
    p.update(over)
    p["episode_length"] = T
    return dict(E=E, N=N, R=R, T=T, seed=seed, action_mix=action_mix, params=p)


def configs() -> dict:
    """BASELINE.json's five configs plus the headline shape and small parity companions."""
    p10 = list(range(1, 11))  # BASELINE.json: integer prices 1..10 (G4)
    big = dict(prices=p10, tax_period=100, thresholds=THRESHOLDS_7, skill_init=SKILL_PARETO_CLIP)
    return {
        # configs[0]: Tiny economy (coin 0, 3 brackets, 11 rate levels, uniform skills)
        "config1_tiny": _cfg(1, 4, 2, 50, 0, prices=p10, tax_period=10, thresholds=[50.0, 100.0],
                             rate_table=rate_table(11), starting_coin=0.0),
        # G38: tiny-dense companion (literal config 1 produces almost no trades)
        "tiny_dense": _cfg(8, 4, 2, 50, 7, prices=p10, tax_period=10, thresholds=[50.0, 100.0],
                           rate_table=rate_table(11), starting_coin=15.0, skill_init=SKILL_PARETO_CLIP,
                           skill_clip_lo=1.0, skill_clip_hi=3.0),
        # configs[1]: paper-scale population
        "config2_paper": _cfg(1024, 100, 2, 1000, 1234, **big),
        # north_star headline: config-2 shape at E=4096
        "headline": _cfg(4096, 100, 2, 1000, 1234, **big),
        # configs[2]: resource scaling
        "config3_resources": _cfg(4096, 100, 6, 1000, 1234, **big),
        # configs[3]: population scaling, 70% market orders, book cap N
        "config4_population": _cfg(256, 1000, 2, 1000, 1234, action_mix="market70", book_cap=1000, **big),
        # configs[4]: on-GPU rollout with the MLP policy (R=3)
        "config5_policy": _cfg(2048, 100, 3, 1000, 1234, action_mix="policy", **big),
        # f3, the paper's section-5 workload: r = 4 / 12 resources (30 / 86 actions), prices {3,6,9}, taxes
        # off, skills ~ N(1,1) that grow by 0.5 % per gather / craft toward 5 (clip [0,5]: G42), R_d = floor(log2 r) (G43)
        "section5_r4": _cfg(4096, 100, 4, 1000, 1234, **section5(4)),
        "section5_r12": _cfg(2048, 100, 12, 1000, 1234, **section5(12)),
    }


def section5(R: int) -> dict:
    """Parameter overrides of the paper's section-5 experiments for R resources."""
    return dict(prices=[3, 6, 9], taxes_enabled=0, skill_init=SKILL_NORMAL_CLIP, skill_mean=1.0, skill_std=1.0,
                skill_clip_lo=0.0, skill_clip_hi=5.0, skill_growth_rate=0.005, skill_max=5.0,
                craft_distinct=max(1, int(math.floor(math.log2(R)))))


def num_actions(R: int, P: int, craft_mode: int, allow_noop: int) -> int:
    return R + (R if craft_mode == CRAFT_PER_RESOURCE else 1) + 2 * R * P + (1 if allow_noop else 0)


def action_probabilities(cfg: dict) -> np.ndarray:
    """Probability of each action index for the synthetic action stream of a config."""
    p = cfg["params"]
    R, P = cfg["R"], len(p["prices"])
    A = num_actions(R, P, p["craft_mode"], p["allow_noop"])
    if cfg["action_mix"] in ("uniform", "policy"):
        return np.full(A, 1.0 / A)
    if cfg["action_mix"] == "market70":
        # BASELINE.json config 4: 70% market orders with prices round(Normal(5,2)) clipped to the grid
        n_craft = R if p["craft_mode"] == CRAFT_PER_RESOURCE else 1
        cdf = lambda x: 0.5 * (1.0 + math.erf((x - 5.0) / (2.0 * math.sqrt(2.0))))
        prices = p["prices"]
        pmf = []
        for k, pr in enumerate(prices):
            lo = -math.inf if k == 0 else pr - 0.5
            hi = math.inf if k == P - 1 else pr + 0.5
            pmf.append((1.0 if hi == math.inf else cdf(hi)) - (0.0 if lo == -math.inf else cdf(lo)))
        pmf = np.array(pmf)
        pmf /= pmf.sum()
        n_other = R + n_craft + (1 if p["allow_noop"] else 0)
        probs = np.zeros(A)
        probs[:R + n_craft] = 0.3 / n_other
        if p["allow_noop"]:
            probs[A - 1] = 0.3 / n_other
        base = R + n_craft
        for side in range(2):
            for r in range(R):
                s = base + side * R * P + r * P
                probs[s:s + P] = 0.7 / (2 * R) * pmf
        return probs
    raise ValueError(cfg["action_mix"])


def action_cdf(cfg: dict) -> np.ndarray:
    """uint32 cumulative thresholds for the rollout-mode generator: action = smallest a with
    x < cdf[a]; the last entry is read as 2^32 by both implementations."""
    probs = action_probabilities(cfg)
    A = len(probs)
    if cfg["action_mix"] in ("uniform", "policy"):
        c = [((a + 1) << 32) // A for a in range(A)]
    else:
        cum = np.cumsum(probs)
        c = [int(math.floor(v * 4294967296.0)) for v in cum]
    c = [min(v, 0xFFFFFFFF) for v in c]
    c[-1] = 0xFFFFFFFF
    return np.array(c, dtype=np.uint32)


def action_stream(cfg: dict, steps: int, seed: int | None = None, E: int | None = None):
    """Seeded per-step population actions [steps][E][N] and government levels [steps][E][B]."""
    E = cfg["E"] if E is None else E
    p = cfg["params"]
    rng = np.random.Generator(np.random.Philox(key=cfg["seed"] if seed is None else seed))
    probs = action_probabilities(cfg)
    A = len(probs)
    if cfg["action_mix"] in ("uniform", "policy"):
        acts = rng.integers(0, A, size=(steps, E, cfg["N"]), dtype=np.int32)
    else:
        acts = rng.choice(A, size=(steps, E, cfg["N"]), p=probs).astype(np.int32)
    B = len(p["thresholds"]) + 1
    gov = rng.integers(0, len(p["rate_table"]), size=(steps, E, B), dtype=np.int32)
    return acts, gov


def _to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round float32 to bfloat16 (nearest even), returned as uint16 bit patterns."""
    b = np.ascontiguousarray(x, np.float32).view(np.uint32).astype(np.uint64)
    return ((b + 0x7FFF + ((b >> 16) & 1)) >> 16).astype(np.uint16)


def policy_dims(cfg: dict) -> dict:
    """Input/output widths of the two policy MLPs of a config."""
    p = cfg["params"]
    R, P, B, L = cfg["R"], len(p["prices"]), len(p["thresholds"]) + 1, len(p["rate_table"])
    return dict(D_pop=6 + 8 * R + B, D_gov=3 * (3 + R) + B + 2, A=num_actions(R, P, p["craft_mode"], p["allow_noop"]),
                gov_out=B * L, B=B, L=L)


def policy_weights(cfg: dict, seed: int = 0, hidden: int = 128, std: float = 0.02, bias_std: float = 0.0):
    """Random-init policy networks of BASELINE.json configs[4]: obs -> 128 -> 128 -> logits, weights
    ~ N(0, std) rounded to bf16 (returned as uint16 bit patterns, [out][in] row-major), biases 0
    (or N(0, bias_std) for tests of the bias path).  Returns (pop_net, gov_net) dicts."""
    d = policy_dims(cfg)
    rng = np.random.Generator(np.random.Philox(key=seed + 77))

    def net(n_in, n_out):
        out = {}
        for name, (o, i) in (("w1", (hidden, n_in)), ("w2", (hidden, hidden)), ("w3", (n_out, hidden))):
            out[name] = _to_bf16_bits((rng.standard_normal((o, i)) * std).astype(np.float32))
        for name, o in (("b1", hidden), ("b2", hidden), ("b3", n_out)):
            out[name] = (rng.standard_normal(o) * bias_std).astype(np.float32)
        return out

    return net(d["D_pop"], d["A"]), net(d["D_gov"], d["gov_out"])
