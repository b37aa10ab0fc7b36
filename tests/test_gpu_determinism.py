"""Race evidence without compute-sanitizer (closed on this pool): the step kernel keeps an economy in shared
memory, aliases the matched-order lists onto the observation staging tile and orders its phases with hand-placed
barriers and bulk-copy waits.  A missing barrier shows up as run-to-run differences, so every workload is run at full
size many times from the same seed -- whole call, split calls, different ring depths, one launch per step -- and
every output of every env must come out bit-identical each time."""
import numpy as np
import pytest

from paper_2410_22165_b200 import binding, inputs

pytestmark = pytest.mark.gpu


def _bits(t):
    import torch
    return t.view(torch.int32) if t.dtype == torch.float32 else t


def _same(a, b, what):
    import torch
    assert torch.equal(_bits(a), _bits(b)), "%s differs between two runs of the same rollout" % what


def _dump(env):
    E = env.E
    return np.concatenate([env.get_state(b, min(512, E - b)) for b in range(0, E, 512)])


@pytest.mark.parametrize("name,T", [("headline", 120), ("config3_resources", 110), ("config4_population", 110), ("section5_r12", 60),
                                    ("config2_paper", 120)])
def test_repeated_full_size_rollouts_are_bit_identical(name, T):
    import torch

    cfg = inputs.configs()[name]
    E, N, R = cfg["E"], cfg["N"], cfg["R"]
    env = binding.Env(E, N, R, cfg["params"])
    env.set_action_cdf(inputs.action_cdf(cfg))
    B = env.B

    def rings(depth):
        return dict(obs_ring=env.new_obs(depth), rew_ring=env.new_rew(depth), done_ring=env.new_done(depth),
                    actions_ring=torch.zeros((depth, E, N), dtype=torch.int32, device="cuda"),
                    gov_actions_ring=torch.zeros((depth, E, B), dtype=torch.int32, device="cuda"))

    # reference: one call, every step kept
    ref = rings(T)
    env.reset(cfg["seed"])
    env.rollout(T, ring_depth=T, **ref)
    torch.cuda.synchronize()
    ref_dump = _dump(env)
    assert (ref_dump[:, 0] == T).all()
    # 1) the same call again and again
    cur = rings(T)
    for rep in range(5):
        for v in cur.values():
            v.fill_(0) if v.dtype != torch.float32 else v.fill_(float("nan"))
        env.reset(cfg["seed"])
        env.rollout(T, ring_depth=T, **cur)
        torch.cuda.synchronize()
        for k in ref:
            _same(cur[k], ref[k], "%s %s (repeat %d)" % (name, k, rep))
        assert np.array_equal(_dump(env), ref_dump), "%s final dump (repeat %d)" % (name, rep)
    del cur
    # 2) split calls with shallow rings: slot s % depth of a call holds its step s
    for chunks, depth in (((T // 2, T - T // 2), 7), ((1, T - 1), 3), ((T // 3, T // 3, T - 2 * (T // 3)), 1)):
        small = rings(depth)
        env.reset(cfg["seed"])
        t0 = 0
        for m in chunks:
            env.rollout(m, ring_depth=depth, **small)
            torch.cuda.synchronize()
            for s in range(max(0, m - depth), m):
                for k in ref:
                    _same(small[k][s % depth], ref[k][t0 + s], "%s %s at t=%d (chunks %s, ring %d)" % (name, k, t0 + s, chunks, depth))
            t0 += m
        assert np.array_equal(_dump(env), ref_dump), "%s final dump (chunks %s)" % (name, chunks)
    # 3) one launch per step through ej_step, fed with the actions the rollout generated
    env.reset(cfg["seed"])
    obs, rew, done = env.new_obs(), env.new_rew(), env.new_done()
    for t in range(T):
        env.step(ref["actions_ring"][t], ref["gov_actions_ring"][t], obs, rew, done)
        if t % 9 == 0 or t == T - 1:
            _same(obs, ref["obs_ring"][t], "%s observations of ej_step at t=%d" % (name, t))
            _same(rew, ref["rew_ring"][t], "%s rewards of ej_step at t=%d" % (name, t))
            _same(done, ref["done_ring"][t], "%s done of ej_step at t=%d" % (name, t))
    torch.cuda.synchronize()
    assert np.array_equal(_dump(env), ref_dump), "%s final dump (ej_step)" % name
