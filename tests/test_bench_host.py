"""Host logic of bench.py that needs no GPU: the algorithmic counts of SURVEY.md §8(d), the per-kernel roofline
arithmetic, and the rule that ncu counters are reported only for the build they were captured on."""
import csv
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
import bench  # noqa: E402


def test_algorithmic_counts_are_the_survey_table():
    """projection 63T + 300, TDI-1 108T + 170, TDI-2 252T + 336 (+ 10 for the A,E,T epilogue);
    1,938 / 2,978 / 6,888 at T = 26 and 2,946 / 10,920 at T = 42; bytes 16 + 48 and 48 + 8 n_out."""
    assert bench.ops_project(26) == 1938 and bench.ops_project(42) == 2946
    assert bench.ops_tdi(26, 1) == 2978 + 10 and bench.ops_tdi(26, 2) == 6888 + 10 and bench.ops_tdi(42, 2) == 10920 + 10
    assert bench.BYTES_PROJECT == 64 and bench.bytes_tdi(3) == 72 and bench.bytes_tdi(6) == 96


def test_kernel_stats_fractions():
    peak, hbm = 1.86e13, 6554.6
    n = 3_153_600.0
    ks = bench.kernel_stats(0.43, 0.32, n, 25, 2, 6, ("fir3", 31, 3), peak, hbm)
    p, t = ks["lr_project"], ks["lr_tdi"]
    assert p["frac_fp64"] == pytest.approx(1938 * n / 0.43e-3 / peak)
    assert p["frac_hbm"] == pytest.approx(64 * n / 0.43e-3 / 1e9 / hbm) and p["bound"] == "alu"
    assert t["executed_ops_per_sample"] == 3 * 4 * 31 * 3 == 1116
    assert t["frac_executed"] == pytest.approx(1116 * n / 0.32e-3 / peak) and t["frac_fp64"] > 1.0
    assert t["bound"] == "alu"
    # order 1: 7 taps -> the filter is nearer its HBM roof than its FP64 roof
    t1 = bench.kernel_stats(0.15, 0.165, n, 1, 2, 6, ("fir3", 7, 3), peak, hbm)["lr_tdi"]
    assert t1["bound"] == "hbm" and t1["frac_hbm"] > t1["frac_executed"]
    # per-sample path: executed = algorithmic
    ps = bench.kernel_stats(0.43, 1.49, n, 25, 2, 6, ("per_sample", 0, 0), peak, hbm)["lr_tdi"]
    assert ps["frac_executed"] == ps["frac_fp64"] and ps["executed_ops_per_sample"] == 6898


def test_ncu_counters_only_for_the_build_they_were_captured_on(tmp_path, monkeypatch):
    path = tmp_path / "counters.csv"
    monkeypatch.setattr(bench, "NCU_COUNTERS", str(path))
    c, why = bench.ncu_counters("year", "lr_project")
    assert c is None and "not found" in why
    row = {k: "" for k in bench.NCU_FIELDS}
    row.update(csrc_sha256="0" * 64, workload="year", api="lr_project", kernel="project_kernel<13, 1>", time_us="440.0",
               registers="128", dram_bytes_read="50000000", dram_bytes_write="97000000", pipe_fp64_pct="70.0",
               smem_wavefronts_pct="84.6", issue_active_pct="50.6", inst_executed="241143658", warps_active_pct="24.1")
    with open(path, "w", newline="") as f:
        wr = csv.DictWriter(f, fieldnames=bench.NCU_FIELDS)
        wr.writeheader()
        wr.writerow(row)
    c, why = bench.ncu_counters("year", "lr_project")
    assert c is None and "csrc/ changed" in why                      # another build: nothing is reported
    c, why = bench.ncu_counters("batch", "lr_project")
    assert c is None and "no ncu capture" in why
    row["csrc_sha256"] = bench.csrc_hash()
    with open(path, "w", newline="") as f:
        wr = csv.DictWriter(f, fieldnames=bench.NCU_FIELDS)
        wr.writeheader()
        wr.writerow(row)
    c, why = bench.ncu_counters("year", "lr_project")
    assert why is None and c["dram_bytes"] == 147000000.0 and c["pipe_fp64_pct"] == 70.0


def test_tracked_counters_match_the_tracked_sources():
    """The committed profiles/r2_ncu_counters.csv belongs to the committed csrc/ (a kernel edit without a new capture
    makes bench.py print null, which is right, but should not be committed unnoticed)."""
    rows = list(csv.DictReader(open(os.path.join(ROOT, "profiles", "r2_ncu_counters.csv"))))
    assert {(r["workload"], r["api"]) for r in rows} >= {("year", "lr_project"), ("year", "lr_tdi"),
                                                         ("batch", "lr_project"), ("batch", "lr_tdi")}
    assert {r["csrc_sha256"] for r in rows} == {bench.csrc_hash()}


def test_ncu_import_reads_a_raw_page(tmp_path, monkeypatch):
    monkeypatch.setattr(bench, "NCU_COUNTERS", str(tmp_path / "out.csv"))
    hdr = ["ID", "Kernel Name", "gpu__time_duration.sum", "launch__registers_per_thread", "dram__bytes_read.sum",
           "dram__bytes_write.sum", "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_elapsed",
           "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed",
           "smsp__issue_active.avg.pct_of_peak_sustained_active", "smsp__inst_executed.sum",
           "sm__warps_active.avg.pct_of_peak_sustained_active"]
    units = ["", "", "us", "register/thread", "Mbyte", "Gbyte", "%", "%", "%", "inst", "%"]
    rows = [["0", "void lr::project_kernel<13, 1>(lr::Params)", "440.5", "128", "50.5", "0.0975", "70", "84", "50", "2.4e8", "24"],
            ["1", "void lr::tdi_fir_apply_kernel<3>(lr::Params)", "323.0", "80", "340", "0.119", "63", "37", "49", "1.7e8", "36"]]
    raw = tmp_path / "raw.csv"
    with open(raw, "w", newline="") as f:
        csv.writer(f).writerows([hdr, units] + rows)
    bench.ncu_import(str(raw), "year")
    got = {r["api"]: r for r in csv.DictReader(open(tmp_path / "out.csv"))}
    assert got["lr_project"]["kernel"] == "project_kernel<13, 1>" and got["lr_project"]["csrc_sha256"] == bench.csrc_hash()
    assert float(got["lr_project"]["dram_bytes_read"]) == 50.5e6 and float(got["lr_project"]["dram_bytes_write"]) == 97.5e6
    assert float(got["lr_tdi"]["time_us"]) == 323.0
