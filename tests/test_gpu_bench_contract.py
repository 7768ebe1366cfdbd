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
