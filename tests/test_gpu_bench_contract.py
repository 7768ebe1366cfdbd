"""bench.py's JSON contract on a GPU (small workload, few steps): one line, the base keys, the tier's `roofline`
and `cpu_baseline` objects, `e2e`, `clocks`, `gpu_launches`; and the `--impl reference` arm."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*args):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                       timeout=900, cwd=ROOT)
    assert r.returncode == 0, r.stdout + r.stderr
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    return json.loads(lines[0])


def test_bench_line_contract():
    d = _run("--gpus", "1", "--steps", "5", "--warmup", "3", "--workload", "tiny", "--peak-seconds", "0.1",
             "--cpu-seconds", "1")
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "roofline", "cpu_baseline", "clocks"):
        assert key in d, key
    assert d["n_gpus"] == 1 and d["steps"] == 5 and d["warmup"] == 3 and d["higher_is_better"] is True
    assert d["dtype"] == "f64" and d["data"] == "synthetic" and d["vs_baseline"] is None
    assert "workload" in d["config"] and "model" not in d["config"]
    assert d["value"] > 0 and d["gpu_launches"] >= 2 * d["steps"]
    rf = d["roofline"]
    for key in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert key in rf, key
    assert rf["bound"] == "alu" and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-12
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] > 0 and cb["sample"]
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    assert e["value"] != d["value"]
    assert {"sm_mhz", "sm_max_mhz", "reasons"} <= set(d["clocks"])


def test_bench_default_line_carries_batch_orders_and_one_thread():
    """The default (one-year) run is the driver's line: besides the contract keys it must carry the batch leg of
    BASELINE.json configs[2] (templates/s, per-kernel fractions), the executed-work fraction of lr_tdi, the order
    sweep and the one-thread oracle figure with the CPU model ("next" item 2)."""
    d = _run("--gpus", "1", "--steps", "3", "--warmup", "3", "--peak-seconds", "0.1", "--cpu-seconds", "1")
    assert d["config"]["workload"].startswith("BASELINE.json configs[1]") and "cached" in d["config"]["tdi_plan"]
    k = d["kernels"]["lr_tdi"]
    assert k["path"] == "fir3" and k["executed_ops_per_sample"] == 3 * 4 * k["fir_taps"] * k["fir_powers"] == 1116
    assert 0.3 < k["frac_executed"] < 1.0 and k["frac_fp64"] > 1.0
    b = d["batch"]
    assert b["templates_per_launch"] == 64 and b["templates_per_s"] > 500 and b["roofline"]["frac"] >= 0.5
    assert b["params_to_loglike"]["loglike_per_s"] > 500
    assert [r["order"] for r in d["orders"]["orders"]] == [1, 9, 25, 41]
    assert all(0 < r[c]["frac"] < 1.2 for r in d["orders"]["orders"] for c in ("lr_project", "lr_tdi"))
    cb = d["cpu_baseline"]
    assert cb["cpu_model"] and cb["one_thread"]["cores"] == 1 and 0 < cb["one_thread"]["value"] < cb["value"]
    rf = d["roofline"]
    assert len(rf["csrc_sha256"]) == 64 and ("unavailable" in rf["ncu"]["lr_project"] or rf["traffic"] > 0)


def test_bench_reference_arm():
    d = _run("--impl", "reference", "--steps", "1", "--warmup", "0", "--workload", "tiny", "--cpu-seconds", "0.5")
    assert d["impl"] == "reference" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


def test_fp64_operand_probe_orders_the_modes(tmp_path):
    """tests/probes/dfma_operand_probe.cu (a test-only translation unit, not part of liblr.so): a DFMA stream that
    shares source registers between neighbours issues faster than one that does not (the measurement behind
    DESIGN.md §6's issue rules), and none exceeds the nominal peak."""
    import ctypes
    import shutil
    import torch
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    so = str(tmp_path / "dfma_operand_probe.so")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-shared", "-Xcompiler", "-fPIC",
                    os.path.join(ROOT, "tests", "probes", "dfma_operand_probe.cu"), "-o", so], check=True)
    L = ctypes.CDLL(so)
    L.probe_fp64_operands.argtypes = [ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    r = []
    for m in range(4):
        v = ctypes.c_double()
        assert L.probe_fp64_operands(m, ctypes.byref(v)) == 0
        r.append(v.value)
    nominal = sms * 64 * 2.2e9
    assert all(0 < x < nominal for x in r), r
    assert r[2] < 0.9 * r[1] and r[1] <= 1.05 * r[0] and r[3] <= 1.02 * r[1], r


def test_shuffle_exchange_is_not_faster_than_lds(tmp_path):
    """tests/probes/shuffle_vs_lds_probe.cu: handing every lane a 16-byte stencil element through warp shuffles
    (4 SHFL.32) delivers no more elements per second than one LDS.128 per lane from shared memory: the measurement
    behind DESIGN.md §6's paragraph on warp shuffles (north_star names them for the stencil reductions; the hot
    kernels read their windows with LDS.128 instead)."""
    import ctypes
    import shutil
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    so = str(tmp_path / "shuffle_vs_lds_probe.so")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-shared", "-Xcompiler", "-fPIC",
                    os.path.join(ROOT, "tests", "probes", "shuffle_vs_lds_probe.cu"), "-o", so], check=True)
    L = ctypes.CDLL(so)
    L.probe_exchange.argtypes = [ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
    r = []
    for m in range(2):
        v = ctypes.c_double()
        assert L.probe_exchange(m, ctypes.byref(v)) == 0
        r.append(v.value)
    print(f"LDS.128: {r[0]:.3e} elements/s, 4 x SHFL.32: {r[1]:.3e} elements/s")
    assert r[0] > 0 and r[1] > 0
    assert r[1] <= 1.05 * r[0], r
