"""ej_rollout_noalloc: the entry point for callers that cannot allocate (its scratch is a static device array) against
the existing path (ej_create + ej_reset + ej_rollout on cudaMalloc'd state), on calls in a row that share the scratch.
Collected last on purpose (pytest -x: a failure here must not hide other tests)."""
import numpy as np
import pytest

from paper_2410_22165_b200 import binding, inputs

pytestmark = pytest.mark.gpu

RTOL, ATOL = 1e-5, 1e-6   # the reward tolerance of tests/parity.py


def _both_paths(name, E, T, seed, over=None):
    import torch

    cfg = inputs.configs()[name]
    params = dict(cfg["params"], **(over or {}))
    N, R = cfg["N"], cfg["R"]
    acts_np, gov_np = inputs.action_stream(dict(cfg, params=params), T, seed=seed, E=E)
    acts, gov = torch.from_numpy(acts_np).cuda(), torch.from_numpy(gov_np).cuda()
    # existing path
    env = binding.Env(E, N, R, params)
    env.reset(seed)
    obs_a, rew_a, done_a = env.new_obs(T), env.new_rew(T), env.new_done(T)
    env.rollout(T, ring_depth=T, actions_in=acts, gov_actions_in=gov, obs_ring=obs_a, rew_ring=rew_a, done_ring=done_a)
    # new entry point: no handle; outputs pre-filled with garbage
    obs_b = torch.full_like(obs_a, float("nan"))
    rew_b = torch.full_like(rew_a, float("nan"))
    done_b = torch.full_like(done_a, 7)
    stream = torch.cuda.current_stream().cuda_stream
    binding.ej_rollout_noalloc(E, N, R, binding.make_params(params), seed, T, acts.data_ptr(), gov.data_ptr(), obs_b.data_ptr(),
                               rew_b.data_ptr(), done_b.data_ptr(), stream)
    torch.cuda.synchronize()
    pop_a, gov_a = env.split_obs(obs_a)
    pop_b, gov_b = env.split_obs(obs_b)
    assert torch.equal(pop_a.view(torch.int32), pop_b.view(torch.int32)), name + ": population observations differ"
    ga, gb = gov_a.cpu().numpy().astype(np.float64), gov_b.cpu().numpy().astype(np.float64)
    assert (np.abs(ga - gb) <= ATOL + RTOL * np.abs(ga)).all(), name + ": government observations differ"
    ra, rb = rew_a.cpu().numpy().astype(np.float64), rew_b.cpu().numpy().astype(np.float64)
    assert np.isfinite(rb).all() and (np.abs(ra - rb) <= ATOL + RTOL * np.abs(ra)).all(), name + ": rewards differ"
    assert torch.equal(done_a, done_b), name + ": done differs"
    return env


def test_noalloc_rollout_equals_the_allocating_path_on_calls_in_a_row():
    # call 1 and 2: the same shape twice with different seeds; call 3: another shape over the same scratch bytes (every
    # call shares the array and must not depend on what the last one left there); call 4: the first call again
    _both_paths("config2_paper", 24, 70, seed=11, over=dict(tax_period=20))
    _both_paths("config2_paper", 24, 70, seed=12, over=dict(tax_period=20))
    _both_paths("config3_resources", 9, 40, seed=5, over=dict(tax_period=10))
    _both_paths("tiny_dense", 8, 55, seed=3)                    # 5 steps past the end of the episode (G28)
    _both_paths("config4_population", 3, 25, seed=2, over=dict(tax_period=10))
    _both_paths("config2_paper", 24, 70, seed=11, over=dict(tax_period=20))


def test_noalloc_limits_and_setup_call():
    import torch

    cfg = inputs.configs()["config2_paper"]
    N, R, p = cfg["N"], cfg["R"], binding.make_params(cfg["params"])
    env = binding.Env(1, N, R, cfg["params"])
    fit = binding.NOALLOC_SCRATCH_BYTES // env.device_state_bytes
    assert fit >= 64
    binding.ej_rollout_noalloc(fit, N, R, p, 1, 0, None, None, None, None, None, None)          # T = 0: set-up only, at the limit
    with pytest.raises(binding.EjError) as ei:                                                    # one env too many
        binding.ej_rollout_noalloc(fit + 1, N, R, p, 1, 0, None, None, None, None, None, None)
    assert ei.value.code == binding.EJ_ERR_PARAM and "static scratch" in str(ei.value) and str(fit) in str(ei.value)
    with pytest.raises(binding.EjError) as ei:                                                    # actions are required
        binding.ej_rollout_noalloc(2, N, R, p, 1, 3, None, None, None, None, None, None)
    assert ei.value.code == binding.EJ_ERR_PARAM and "actions" in str(ei.value)
    with pytest.raises(binding.EjError) as ei:                                                    # parameter validation as in ej_create
        binding.ej_rollout_noalloc(2, N, R, binding.make_params(dict(cfg["params"], eta=1.0)), 1, 0, None, None, None, None, None, None)
    assert "eta" in str(ei.value)
    torch.cuda.synchronize()
