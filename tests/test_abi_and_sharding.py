"""CPU-side checks: the C-ABI library loads and exports every symbol include/econojax.h declares,
the ctypes structs have the sizes the C compiler gives the header's structs, the library fails
loudly without a GPU, and the N > 1 sharding logic (gloo, world size 2)."""
import ctypes as C
import os
import re
import subprocess
import sys
import tempfile

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HDR = os.path.join(ROOT, "include", "econojax.h")


def declared_symbols():
    src = open(HDR).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ej_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_2410_22165_b200 import binding

    names = declared_symbols()
    assert {"ej_create", "ej_reset", "ej_step", "ej_rollout", "ej_set_policy", "ej_policy_act"} <= set(names)
    L = binding.lib()
    for n in names:
        assert hasattr(L, n), "libeconojax.so does not export %s" % n
    assert set(binding.EXPORTS) == set(names)


def test_ctypes_structs_match_the_header():
    from paper_2410_22165_b200 import binding

    prog = '#include <stdio.h>\n#include "econojax.h"\nint main(void){printf("%zu %zu %zu %zu\\n", sizeof(ej_params), sizeof(ej_layout_info), sizeof(ej_rollout_io), sizeof(ej_mlp));return 0;}\n'
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "s.c")
        open(c, "w").write(prog)
        exe = os.path.join(d, "s")
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), "-o", exe, c])
        sizes = [int(x) for x in subprocess.check_output([exe]).split()]
    assert sizes == [C.sizeof(binding.EjParams), C.sizeof(binding.EjLayoutInfo), C.sizeof(binding.EjRolloutIO), C.sizeof(binding.EjMlp)]


def test_no_cpu_fallback():
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2410_22165_b200 import binding, inputs

    cfg = inputs.configs()["tiny_dense"]
    with pytest.raises(binding.EjError) as ei:
        binding.ej_create(1, cfg["N"], cfg["R"], binding.make_params(cfg["params"]))
    assert ei.value.code == binding.EJ_ERR_CUDA and "no CPU fallback" in str(ei.value)


def test_parameter_validation_names_the_field():
    from paper_2410_22165_b200 import binding, inputs

    cfg = inputs.configs()["tiny_dense"]
    for field, value, expect in (("prices", [3, 2, 1], "prices"), ("eta", 1.0, "eta"), ("max_active_orders", 99, "max_active_orders"),
                                 ("thresholds", [5.0, 4.0], "thresholds")):
        with pytest.raises(binding.EjError) as ei:
            binding.ej_create(1, cfg["N"], cfg["R"], binding.make_params(dict(cfg["params"], **{field: value})))
        assert ei.value.code == binding.EJ_ERR_PARAM and expect in str(ei.value)


def _worker(rank, world, port, q):
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import oracle
    from paper_2410_22165_b200 import inputs, sharding

    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    cfg = inputs.configs()["tiny_dense"]
    E = 3
    base = sharding.shard_env_base(rank, world, E)
    bases = [None] * world
    dist.all_gather_object(bases, base)
    # the shard a rank would hand to ej_create: the oracle stands in for the device here, keyed the same way
    o = oracle.OracleEnv(E, cfg["N"], cfg["R"], dict(cfg["params"], env_id_base=base))
    o.reset(cfg["seed"])
    acts, gov = inputs.action_stream(cfg, 20, seed=3, E=E * world)
    for t in range(20):
        o.step(acts[t][base:base + E], gov[t][base:base + E], want_obs=False)
    states = [None] * world
    dist.all_gather_object(states, o.get_state())
    tmax = sharding.max_over_ranks(10.0 + rank, dist)
    dist.barrier()
    dist.destroy_process_group()
    if rank == 0:
        q.put((bases, np.concatenate(states), tmax, sharding.total_units(E * cfg["N"] * 20, world)))


def test_sharded_run_equals_unsharded_gloo_world2():
    import torch.multiprocessing as mp

    sys.path.insert(0, ROOT)
    import oracle
    from paper_2410_22165_b200 import inputs

    world, port = 2, 29500 + os.getpid() % 2000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    bases, states, tmax, units = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert bases == [0, 3] and tmax == 11.0 and units == 2 * 3 * 4 * 20
    cfg = inputs.configs()["tiny_dense"]
    o = oracle.OracleEnv(6, cfg["N"], cfg["R"], cfg["params"])
    o.reset(cfg["seed"])
    acts, gov = inputs.action_stream(cfg, 20, seed=3, E=6)
    for t in range(20):
        o.step(acts[t], gov[t], want_obs=False)
    assert np.array_equal(states, o.get_state())
