"""CPU-side checks (no GPU): the C-ABI library builds, loads and exports every symbol include/lr.h
declares; host-only entry points behave; the batch sharding used for N > 1 GPUs is a partition."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2204_06633_b200 import binding, build
    build.build()
    return binding.lib()


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "lr.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lr_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_exported(lib):
    from paper_2204_06633_b200 import binding
    decl = _declared_symbols()
    assert sorted(binding.SYMBOLS) == decl
    for name in decl:
        assert hasattr(lib, name), f"liblr.so does not export {name}"


def test_header_compiles_as_c():
    """include/lr.h is plain C: no torch or C++ types in the signatures."""
    code = '#include "lr.h"\nint main(void){ lr_orbits o; (void)o; return LR_MAX_ORDER == 65 ? 0 : 1; }\n'
    r = subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-fsyntax-only", "-I", os.path.join(ROOT, "include"),
                        "-x", "c", "-"], input=code, text=True, capture_output=True)
    assert r.returncode == 0, r.stderr


def test_host_only_entry_points(lib):
    from paper_2204_06633_b200 import binding
    assert binding.lr_strerror(0) == "success"
    for code in (-1, -2, -3, -4, -99):
        assert binding.lr_strerror(code)
    assert binding.lr_launch_count() >= 0
    # argument validation happens before any CUDA call
    h = ctypes.c_void_p()
    assert lib.lr_create(None, 10.0, 25, 2, ctypes.byref(h)) == binding.LR_EINVAL
    assert lib.lr_set_option(None, 1, 0.0) == binding.LR_EINVAL
    assert lib.lr_get_margins(None, None, None, None) == binding.LR_EINVAL
    assert lib.lr_project(None, None, None, None, None, None, 1, 1, None, None) == binding.LR_EINVAL
    assert lib.lr_tdi(None, None, 1, 1, None, None) == binding.LR_EINVAL
    lib.lr_destroy(None)


def test_gb_parameters_host(lib):
    """lr_gb_parameters (host arithmetic of eqs. 8-9) against the oracle's statement of the same equations."""
    from oracle import waveform as owf
    from paper_2204_06633_b200 import binding
    A, f0, fdot, phi0, iota = 1.3e-22, 4.2e-3, 2.5e-16, 0.9, 1.1
    g = binding.lr_gb_parameters(A, f0, fdot, phi0, iota, binding.LR_GB_PAPER)
    ap, ac = owf.amplitudes_paper(A, iota)
    assert np.allclose(g, [ap, ac, f0, fdot, owf.fddot_eq8(f0, fdot), phi0], rtol=1e-15, atol=0)
    g = binding.lr_gb_parameters(A, f0, fdot, phi0, iota, binding.LR_GB_CONFIG)
    ap, ac = owf.amplitudes_config(A, iota)
    assert np.allclose(g, [ap, ac, f0, fdot, 0.0, phi0], rtol=1e-15, atol=0)
    for bad in ((A, 0.0, fdot, phi0, iota, 0), (A, f0, fdot, phi0, iota, 7), (float("nan"), f0, fdot, phi0, iota, 0)):
        with pytest.raises(binding.LrError):
            binding.lr_gb_parameters(*bad)


def test_create_rejects_bad_arguments_without_gpu(lib):
    from harness import inputs
    from paper_2204_06633_b200 import binding
    tab = inputs.orbit_table("eq", 0.0, 86400.0)
    for order, gen, dt in ((24, 2, 10.0), (0, 2, 10.0), (67, 2, 10.0), (25, 3, 10.0), (25, 2, 0.0)):
        with pytest.raises(binding.LrError) as e:
            binding.lr_create(tab, dt, order, gen)
        assert e.value.code == binding.LR_EINVAL
    bad = inputs.OrbitTable(tab.t_start, tab.knot_dt, tab.x.copy(), tab.ltt.copy())
    bad.x[0, 0, 1] = np.nan
    with pytest.raises(binding.LrError):
        binding.lr_create(bad, 10.0, 25, 2)


def test_no_cpu_fallback_without_device(lib):
    """Without a CUDA device a valid lr_create fails with LR_ECUDA: there is no CPU compute path."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from harness import inputs
    from paper_2204_06633_b200 import binding
    tab = inputs.orbit_table("eq", 0.0, 86400.0)
    with pytest.raises(binding.LrError) as e:
        binding.lr_create(tab, 10.0, 25, 2)
    assert e.value.code == binding.LR_ECUDA


def test_product_never_imports_oracle():
    """The product path shares nothing with oracle/ (and does not read _work/)."""
    pkg = os.path.join(ROOT, "paper_2204_06633_b200")
    for dirpath, _, files in os.walk(pkg):
        if os.path.basename(dirpath) == "build":
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".hpp", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, flags=re.M), f
                assert "lr_oracle" not in text and "_work/" not in text, f
    text = open(os.path.join(ROOT, "oracle", "lr_oracle.cpp")).read()
    assert "paper_2204_06633_b200/csrc/" not in re.sub(r"//.*", "", text)


def test_shard_templates_is_a_partition():
    from paper_2204_06633_b200 import shard_templates
    for batch in (0, 1, 7, 128, 1024, 1025):
        for world in (1, 2, 3, 8):
            spans = [shard_templates(batch, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == batch
            for a, b in zip(spans, spans[1:]):
                assert a[1] == b[0]
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_templates(4, 2, 2)


def test_shard_time_is_a_partition_with_halos():
    from paper_2204_06633_b200 import shard_time
    unit, lo, hi = 1792, 90, 87
    for n in (1, 1791, 1792, 10640, 3153600):
        for world in (1, 2, 3, 8):
            spans = [shard_time(n, r, world, unit, lo, hi) for r in range(world)]
            pos = 0
            for first, count, h_first, h_len in spans:
                if count == 0:
                    assert h_len == 0
                    continue
                assert first == pos and first % unit == 0
                assert h_first == max(0, first - lo) and h_first + h_len == min(n, first + count + hi)
                pos = first + count
            assert pos == n
    with pytest.raises(ValueError):
        shard_time(10, 3, 2, unit, lo, hi)


_GLOO_WORKER = r'''
import os, sys
sys.path.insert(0, sys.argv[1])
import torch, torch.distributed as dist
from paper_2204_06633_b200 import gather_scalars, shard_templates, shard_time
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
batch = 11
lo, hi = shard_templates(batch, rank, world)
# every rank claims its templates; the union must be a partition (no data-path collective is involved)
own = torch.zeros(batch, dtype=torch.int64); own[lo:hi] = 1
dist.all_reduce(own)
assert bool((own == 1).all()), own
# time-axis sharding of one long template: the ranks' spans tile [0, n) (halos are recomputed, not exchanged)
n = 100000
first, count, h_first, h_len = shard_time(n, rank, world, 1792, 90, 87)
cover = torch.zeros(n, dtype=torch.int64); cover[first:first + count] = 1
dist.all_reduce(cover)
assert bool((cover == 1).all())
# the likelihood stage's only exchange: all-gather of the per-template scalars, unequal shards (11 over 2 ranks)
mine = torch.arange(lo, hi, dtype=torch.float64) * 1.5 - 7.0
full = gather_scalars(mine, batch, rank, world)
assert torch.equal(full, torch.arange(batch, dtype=torch.float64) * 1.5 - 7.0), full
# max-over-ranks timing + whole-job aggregation used by bench.py
ms = bench.max_over_ranks(10.0 * (rank + 1))
assert ms == 10.0 * world, ms
tot = bench.sum_over_ranks(float(hi - lo))
assert tot == batch, tot
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
'''


def test_multi_rank_host_logic_gloo(tmp_path):
    """world_size-2 run of the N > 1 host logic on CPU (gloo): template sharding partitions the batch,
    timing is the max over ranks, units are summed over ranks."""
    script = tmp_path / "worker.py"
    script.write_text(_GLOO_WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                        "--master-addr", "127.0.0.1", "--master-port", "29517", str(script), ROOT],
                       capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0, r.stdout + r.stderr
    assert r.stdout.count("ok") == 2


def test_bench_reference_arm_two_ranks():
    """`bench.py --impl reference` under torchrun with 2 ranks: rank 0 alone times the oracle and prints ONE
    JSON line with the contract's keys; the other rank exits 0 without work."""
    import json
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                        "--master-addr", "127.0.0.1", "--master-port", "29519", os.path.join(ROOT, "bench.py"),
                        "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--workload", "tiny",
                        "--cpu-seconds", "0.5"], capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stdout + r.stderr
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    for key in ("metric", "unit", "steps", "warmup", "ms_per_step", "higher_is_better", "config", "cpu_baseline", "e2e"):
        assert key in d, key
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
