"""CPU-side tests: the C-ABI library builds, loads and exports every symbol include/chisao.h declares;
host-only entry points validate their arguments; the multi-GPU host logic (independent replicas) works
over gloo with world_size 2.  No compute call is made here (no GPU in this container)."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

from paper_2606_26164_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_26164_b200 import build, binding
    build.build()
    return binding.load_library()


def test_library_exports_every_declared_symbol(lib):
    from paper_2606_26164_b200 import binding
    header = open(os.path.join(ROOT, "include", "chisao.h")).read()
    declared = set(re.findall(r"CHISAO_API[^;(]*?(chisao_[a-z_]+)\s*\(", header))
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    # nothing of the oracle is linked in, and the CUDA runtime is linked statically
    out = subprocess.run(["nm", "-D", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "orc_" not in out


def test_workspace_bytes_is_host_only_and_scales(lib):
    from paper_2606_26164_b200 import binding
    small = binding.workspace_bytes(inputs.config(5, N=1024))
    big = binding.workspace_bytes(inputs.config(5))
    assert small > 0 and big > 300e6 and big < 2e9            # history alone is 2*m*N*d*4 = 335 MB at C5
    hist = 2 * 10 * 65536 * 64 * 4
    assert big > hist
    assert binding.workspace_bytes(inputs.custom(inputs.gmm_iso(2, 2, 0.3, 1.0, 3), 2.0, 0)) > 0


def test_invalid_configurations_are_rejected_without_a_device(lib):
    from paper_2606_26164_b200 import binding
    wl = inputs.config(1)
    for field, bad in (("d", 0), ("d", 65), ("lbfgs_m", 0), ("lbfgs_m", 17), ("hlc_M", 0), ("ls_max", -1),
                       ("reseed_cands", 17), ("n_osc", 0), ("sigma_s", 0.0)):
        cfg, obj, keep = binding.marshal(wl)
        setattr(cfg, field, bad)
        if field == "d":
            obj.d = bad
        n = C.c_size_t(0)
        assert lib.chisao_workspace_bytes(C.byref(cfg), C.byref(obj), C.byref(n)) == binding.E_INVALID, field
        assert len(lib.chisao_last_error(None)) > 0
    cfg, obj, keep = binding.marshal(wl)
    obj.id = 9
    n = C.c_size_t(0)
    assert lib.chisao_workspace_bytes(C.byref(cfg), C.byref(obj), C.byref(n)) == binding.E_INVALID
    assert lib.chisao_step(None, None) == binding.E_INVALID
    assert lib.chisao_launch_count(None) == 0
    lib.chisao_destroy(None)


def test_binding_refuses_to_run_without_cuda():
    import torch
    from paper_2606_26164_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(RuntimeError):
        binding.Chisao(inputs.config(1))


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_26164_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "chisao_oracle" not in src and "liboracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "libchisao" not in src and "include/chisao.h\"" not in src and "binding" not in src, f


def test_replica_workloads_differ_only_in_seeds():
    from paper_2606_26164_b200 import replicas
    a, b = replicas.replica_workload(2, 0, N=64), replicas.replica_workload(2, 1, N=64)
    assert np.array_equal(a.obj.means, b.obj.means) and a.hp.seed != b.hp.seed
    assert not np.array_equal(a.x0, b.x0)
    assert np.array_equal(a.x0, inputs.config(2, N=64).x0)


_WORKER = r"""
import os, sys
sys.path.insert(0, sys.argv[1])
import torch.distributed as dist
from paper_2606_26164_b200 import replicas
dist.init_process_group("gloo")
r = dist.get_rank()
wl = replicas.replica_workload(1, r, N=32)
mx = replicas.max_over_ranks(10.0 + r, dist)
sm = replicas.sum_over_ranks(float(wl.hp.seed), dist)
assert mx == 11.0, mx
assert sm == (3001) + (3001 + 100000), sm
dist.barrier()
dist.destroy_process_group()
print("ok", r)
"""


def test_replica_reductions_over_gloo_world_size_2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", "29517", str(script), ROOT]
    res = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=240)
    assert res.returncode == 0, res.stderr[-2000:]
    assert res.stdout.count("ok") == 2


def test_bench_gpus_2_self_launches_two_ranks_and_rank_0_prints_one_line():
    """`python bench.py --gpus 2` with no launcher around it starts two ranks itself (bench.py: self_launch); the
    reference arm needs no GPU, so the launch path is checked here: rank 0 prints the one JSON line with n_gpus = 2,
    rank 1 exits 0 without output."""
    import json
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_PORT")}
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference", "--config", "1",
           "--steps", "3", "--warmup", "1"]
    res = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=300, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, res.stdout[-2000:]
    rec = json.loads(lines[0])
    assert rec["n_gpus"] == 2 and rec["impl"] == "reference" and rec["scaling"] == "weak"
    assert rec["value"] > 0 and rec["e2e"]["h2d_bytes_per_step"] == 0
