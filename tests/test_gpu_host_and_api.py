"""GPU tests of the host-buffer step (ej_step_host: the call bench.py's e2e number is timed through) and of the
handle life-cycle corners of the C ABI: kernels shared by handles of different shapes, ej_set_state's preconditions,
pointer alignment."""
import numpy as np
import pytest

import oracle
from paper_2410_22165_b200 import binding, inputs
from parity import Pair, close, compare_outputs, compare_state, exact

pytestmark = pytest.mark.gpu


def _split_host_obs(g, obs):
    pop = obs[: g.E * g.N * g.D_pop].reshape(g.E, g.N, g.D_pop)
    gov = obs[g.gov_obs_offset:].reshape(g.E, g.D_gov_pad)[:, : g.D_gov]
    return pop, gov


@pytest.mark.parametrize("name,E,over", [("config2_paper", 5, dict(tax_period=10)), ("config3_resources", 3, dict(tax_period=15)),
                                         ("tiny_dense", 8, {}), ("config4_population", 1, dict(tax_period=8))])
def test_step_host_dense_against_the_oracle(name, E, over):
    """ej_step_host with pageable and with pinned host buffers, every output column against the oracle; optional
    outputs left NULL on some steps."""
    import torch

    cfg = inputs.configs()[name]
    params = dict(cfg["params"], **over)
    N = cfg["N"]
    pair = Pair(E, N, cfg["R"], params, 6)
    g = pair.g
    T = 32
    acts, gov = inputs.action_stream(dict(cfg, params=params), T, seed=6, E=E)
    pageable = (np.zeros(g.obs_floats, np.float32), np.zeros((E, N + 1), np.float32), np.zeros(E, np.uint8))
    pinned_t = (torch.zeros(g.obs_floats, dtype=torch.float32).pin_memory(), torch.zeros((E, N + 1), dtype=torch.float32).pin_memory(),
                torch.zeros(E, dtype=torch.uint8).pin_memory())
    pinned = tuple(t.numpy() for t in pinned_t)
    for t in range(T):
        obs, rew, done = pinned if t % 2 else pageable
        mode = t % 4
        o_pop, o_gov, o_rew, o_done = pair.o[0].step(acts[t], gov[t])
        if mode == 3:      # rewards only
            rew[:] = -7.0
            g.step_host(acts[t], gov[t], None, rew, None)
            close(rew, o_rew, "%s t=%d rewards (only output)" % (name, t))
        elif mode == 2:    # int64 actions as numpy makes them by default: converted, not reinterpreted
            obs[:] = -7.0
            g.step_host(acts[t].astype(np.int64), gov[t].astype(np.int64), obs, None, done)
            pop, gv = _split_host_obs(g, obs)
            exact(pop, o_pop, "%s t=%d population observations" % (name, t))
            exact(done, o_done, "%s t=%d done" % (name, t))
        else:
            obs[:] = -7.0
            rew[:] = -7.0
            done[:] = 9
            g.step_host(acts[t], gov[t], obs, rew, done)
            pop, gv = _split_host_obs(g, obs)
            compare_outputs(g, pop, gv, rew, done, o_pop, o_gov, o_rew, o_done, "%s t=%d" % (name, t))
    compare_state(pair.g_state(), pair.o_state(), name + " state after host steps")
    with pytest.raises(AssertionError):
        g.step_host(acts[0], gov[0], np.zeros(g.obs_floats, np.float64), None, None)      # wrong dtype of an output buffer
    with pytest.raises(AssertionError):
        g.step_host(acts[0][:, :-1], gov[0], None, None, None)                             # wrong size of an input


def test_handles_of_different_shapes_share_kernels():
    """The reset / observe / generic step kernels are shared by every handle with the same CTA size, while the
    shared memory they need depends on R, P, M: creating a smaller handle must not take memory away from an older,
    larger one (the per-function attribute is only ever raised)."""
    import torch

    big = inputs.configs()["section5_r12"]            # R = 12: ~72 KB of shared memory, 128-thread CTAs
    small = inputs.configs()["config2_paper"]         # R = 2: ~28 KB, same CTA size and stride
    tiny = dict(small["params"], prices=[2, 4], max_active_orders=3)
    a = Pair(3, big["N"], big["R"], big["params"], 3)
    b = Pair(2, small["N"], small["R"], small["params"], 3)
    c = Pair(2, small["N"], small["R"], tiny, 3)      # generic kernels at R = 2 with an even smaller layout
    assert a.g.smem_bytes > b.g.smem_bytes > c.g.smem_bytes
    for pair, cfg, params in ((a, big, big["params"]), (c, small, tiny), (b, small, small["params"]), (a, big, big["params"])):
        pair.g.reset(3)
        pair.o[0].reset(3)
        acts, gov = inputs.action_stream(dict(cfg, params=params), 6, seed=1, E=pair.g.E)
        for t in range(6):
            pair.step_and_compare(acts[t], gov[t], "shared kernels t=%d" % t, check_state=(t == 5))
        pop, gv = pair.g.split_obs(pair.g.observe())
        exact(pop.cpu().numpy(), pair.o[0].observe()[0], "observe after another handle was created")
        pair.g.rollout(5)
    torch.cuda.synchronize()


def test_set_state_preconditions():
    cfg = inputs.configs()["tiny_dense"]
    N, R, p = cfg["N"], cfg["R"], cfg["params"]
    src = oracle.OracleEnv(2, N, R, p)
    src.reset(4)
    acts, gov = inputs.action_stream(cfg, 12, seed=4, E=2)
    for t in range(12):
        src.step(acts[t], gov[t], want_obs=False)
    w = src.get_state()
    fresh = binding.Env(2, N, R, p)
    with pytest.raises(binding.EjError) as ei:       # the dump holds no Philox key: reset (with the run's seed) first
        fresh.set_state(w)
    assert ei.value.code == binding.EJ_ERR_STATE and "ej_reset" in str(ei.value)
    fresh.reset(4)
    fresh.set_state(w[1:2], env_begin=1)             # a sub-range leaves the other env as reset made it
    ref = binding.Env(2, N, R, p)
    ref.reset(4)
    exact(fresh.get_state(0, 1), ref.get_state(0, 1), "env outside the restored range")
    exact(fresh.get_state(1, 1)[:, :11], w[1:2, :11], "restored env")
    exact(fresh.get_state(1, 1)[:, 13:], w[1:2, 13:], "restored env")
    # a crossed book (best bid >= best ask) can never rest (G13): rejected, the state stays as it was
    s = oracle.parse_state(w[0])
    q = 13 + s["B"] + R + N * (6 + 3 * R)
    bad = w[0:1].copy()
    cap = s["cap"]
    bad[0, q] = 1
    bad[0, q + 1:q + 4] = [9, 0, 0]                  # bid of agent 0 at 9 ...
    bad[0, q + 1 + 3 * cap] = 1
    bad[0, q + 2 + 3 * cap:q + 5 + 3 * cap] = [4, 1, 0]   # ... against an ask of agent 1 at 4
    before = fresh.get_state()
    with pytest.raises(binding.EjError) as ei:
        fresh.set_state(bad)
    assert ei.value.code == binding.EJ_ERR_PARAM and "crossed" in str(ei.value)
    exact(fresh.get_state(), before, "state after a rejected ej_set_state")


def test_misaligned_pointers_are_rejected():
    import torch

    cfg = inputs.configs()["config2_paper"]
    env = binding.Env(2, cfg["N"], cfg["R"], cfg["params"])
    env.reset(1)
    acts = torch.zeros((2, cfg["N"]), dtype=torch.int32, device="cuda")
    gov = torch.zeros((2, env.B), dtype=torch.int32, device="cuda")
    buf = torch.zeros(env.obs_floats + 4, dtype=torch.float32, device="cuda")
    rew = env.new_rew()
    for off in (1, 2, 3):
        with pytest.raises(binding.EjError) as ei:
            binding.ej_step(env.h, acts.data_ptr(), gov.data_ptr(), buf.data_ptr() + 4 * off, rew.data_ptr(), None)
        assert ei.value.code == binding.EJ_ERR_PARAM and "aligned" in str(ei.value)
        with pytest.raises(binding.EjError):
            binding.ej_observe(env.h, buf.data_ptr() + 4 * off)
        with pytest.raises(binding.EjError):
            env.rollout(2, obs_ring=buf[off:off + env.obs_floats].unsqueeze(0))
    with pytest.raises(binding.EjError):
        binding.ej_step(env.h, acts.data_ptr(), gov.data_ptr(), None, rew.data_ptr() + 2, None)
    binding.ej_step(env.h, acts.data_ptr(), gov.data_ptr(), buf.data_ptr() + 16, rew.data_ptr(), None)   # aligned: accepted
    torch.cuda.synchronize()
    assert env.get_state()[0, 0] == 1                 # only the accepted call stepped
