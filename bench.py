#!/usr/bin/env python
"""bench.py — response samples/s of the LISA response hot path (lr_project + lr_tdi) on B200.

Contract: `python bench.py --gpus N --steps K --warmup W` prints ONE JSON line.
  * a step = one pass of the whole hot path (six-link projection + TDI-2) over one batch of synthetic input;
  * N = 1 workload = BASELINE.json configs[1]: one Galactic binary, 1 year at dt = 10 s (3,153,600 samples),
    Keplerian orbits, Lagrange order 25, nested second-generation TDI, X,Y,Z + A,E,T;
  * the default run also carries a `batch` leg (one 64-template launch of configs[2], the MCMC batch: templates/s,
    per-kernel roofline fractions, clocks, parameters -> log L) and an `orders` leg (orders 1, 9, 25, 41 on the
    one-year shape: ms and fraction of the binding roof per kernel); `--workload batch` times all 1,024 templates;
  * N > 1: every rank runs the same-sized workload on its own seeded template(s) (the path shards over
    templates with no collective: "scaling": "weak"); time = max over ranks, value = all ranks' samples / time;
  * `value` has the inputs resident in HBM; `e2e` goes through lr_response_host with pinned HOST buffers;
  * `roofline`: the dominant kernel (the slower of lr_project / lr_tdi) against the FP64 issue rate measured
    live by lr_measure_fp64_peak; `kernels` has both, lr_tdi also against the FMAs its FIR path EXECUTES;
  * ncu-only counters (DRAM traffic, pipe busy) come from profiles/r2_ncu_counters.csv and are reported only while
    the hash of csrc/ recorded there equals the sources this run was built from (null + reason otherwise);
  * `cpu_baseline` / `--impl reference`: the oracle (fp64 arithmetic) on a bounded sample, all host cores and one.
"""
from __future__ import annotations

import argparse
import csv
import hashlib
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
DEFAULT_CHUNK = 64   # templates per launch of the batched config (tests/test_gpu_fullsize.py checks this shape)
NCU_COUNTERS = os.path.join(ROOT, "profiles", "r2_ncu_counters.csv")
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def csrc_hash():
    """sha256 over the sources liblr.so is built from (names and contents, sorted): the key of the ncu counters."""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2204_06633_b200", "csrc")
    for name in sorted(os.listdir(d)) + [os.path.join("..", "..", "include", "lr.h")]:
        path = os.path.join(d, name)
        if os.path.isfile(path) and name.endswith((".cu", ".cuh", ".hpp", ".h")):
            h.update(os.path.basename(name).encode())
            h.update(open(path, "rb").read())
    return h.hexdigest()


def ncu_counters(workload, kernel):
    """Counters of one `ncu --set full` capture (profiles/r2_ncu_counters.csv; the .md beside it names the command),
    valid only for the build they were captured on.  Returns (dict or None, reason)."""
    try:
        rows = list(csv.DictReader(open(NCU_COUNTERS)))
    except OSError:
        return None, "profiles/r2_ncu_counters.csv not found"
    rows = [r for r in rows if r["workload"] == workload and r["api"] == kernel]
    if not rows:
        return None, f"no ncu capture of {kernel} on the {workload} workload"
    now = csrc_hash()
    r = rows[-1]
    if r["csrc_sha256"] != now:
        return None, f"csrc/ changed since the capture (captured {r['csrc_sha256'][:12]}, built from {now[:12]})"
    num = lambda k: float(r[k]) if r.get(k) not in (None, "") else None
    return {"kernel": r["kernel"], "time_us": num("time_us"), "dram_bytes": num("dram_bytes_read") + num("dram_bytes_write"),
            "pipe_fp64_pct": num("pipe_fp64_pct"), "smem_wavefronts_pct": num("smem_wavefronts_pct"),
            "issue_active_pct": num("issue_active_pct"), "registers": num("registers"),
            "pipe_dmma_pct": num("pipe_dmma_pct")}, None


# algorithmic FP64 instruction slots per time sample (SURVEY.md §8(d), T = order + 1 taps; DFMA = 1)
NCU_FIELDS = ("csrc_sha256", "workload", "api", "kernel", "time_us", "registers", "dram_bytes_read", "dram_bytes_write",
              "pipe_fp64_pct", "smem_wavefronts_pct", "issue_active_pct", "inst_executed", "warps_active_pct", "pipe_dmma_pct")


def ncu_import(raw_csv, workload):
    """`bench.py --ncu-import FILE --ncu-workload W`: FILE is `ncu -i X.ncu-rep --page raw --csv` of a full capture of
    `bench.py`; takes the LAST captured launch of each of the two hot kernels and (re)writes their rows for workload W
    in profiles/r2_ncu_counters.csv under the hash of the current csrc/.  Runs without a GPU."""
    rows = list(csv.reader(open(raw_csv)))
    hdr, body = rows[0], [r for r in rows[2:] if len(r) == len(rows[0])]
    ix = {h: i for i, h in enumerate(hdr)}
    unit = dict(zip(hdr, rows[1]))

    def val(r, key, scale=None):
        v = float(r[ix[key]].replace(",", ""))
        u = unit.get(key, "")
        if key.startswith("dram__bytes"):
            v *= {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}[u]
        if key == "gpu__time_duration.sum":
            v *= {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}.get(u, 1e-3)   # -> us
        return v

    new = []
    for api, pat in (("lr_project", "project_kernel"), ("lr_tdi", "tdi_fir_apply")):
        hits = [r for r in body if pat in r[ix["Kernel Name"]]]
        if not hits:
            continue
        r = hits[-1]
        new.append({"csrc_sha256": csrc_hash(), "workload": workload, "api": api,
                    "kernel": r[ix["Kernel Name"]].split("(")[0].replace("void ", "").replace("lr::", ""),
                    "time_us": f"{val(r, 'gpu__time_duration.sum'):.1f}",
                    "registers": r[ix["launch__registers_per_thread"]],
                    "dram_bytes_read": f"{val(r, 'dram__bytes_read.sum'):.0f}",
                    "dram_bytes_write": f"{val(r, 'dram__bytes_write.sum'):.0f}",
                    "pipe_fp64_pct": f"{val(r, 'sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_elapsed'):.2f}",
                    "smem_wavefronts_pct": f"{val(r, 'l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed'):.2f}",
                    "issue_active_pct": f"{val(r, 'smsp__issue_active.avg.pct_of_peak_sustained_active'):.2f}",
                    "inst_executed": f"{val(r, 'smsp__inst_executed.sum'):.0f}",
                    "warps_active_pct": f"{val(r, 'sm__warps_active.avg.pct_of_peak_sustained_active'):.2f}",
                    "pipe_dmma_pct": (f"{val(r, 'sm__pipe_tensor_subpipe_dmma_cycles_active.avg.pct_of_peak_sustained_active'):.2f}"
                                      if "sm__pipe_tensor_subpipe_dmma_cycles_active.avg.pct_of_peak_sustained_active" in ix else "")})
    old = []
    if os.path.exists(NCU_COUNTERS):
        old = [r for r in csv.DictReader(open(NCU_COUNTERS)) if not (r["workload"] == workload and r["api"] in {n["api"] for n in new})]
    with open(NCU_COUNTERS, "w", newline="") as f:
        wr = csv.DictWriter(f, fieldnames=NCU_FIELDS)
        wr.writeheader()
        for r in old + new:
            wr.writerow({k: r.get(k, "") for k in NCU_FIELDS})
    print(f"wrote {len(new)} rows for workload {workload} to {NCU_COUNTERS}")


def ops_project(T):
    return 63 * T + 300


def ops_tdi(T, gen):
    return (252 * T + 336 if gen == 2 else 108 * T + 170) + 10


# algorithmic HBM bytes per time sample
BYTES_PROJECT = 16 + 48


def bytes_tdi(nout):
    return 48 + 8 * nout


# ------------------------------------------------------------------------------------------ distributed
def _dist():
    import torch.distributed as dist
    return dist if dist.is_available() and dist.is_initialized() else None


def _reduce(x, op):
    import torch
    dist = _dist()
    if dist is None:
        return float(x)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(x)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=op)
    return float(t.item())


def max_over_ranks(x):
    import torch.distributed as dist
    return _reduce(x, dist.ReduceOp.MAX)


def sum_over_ranks(x):
    import torch.distributed as dist
    return _reduce(x, dist.ReduceOp.SUM)


def barrier():
    dist = _dist()
    if dist is not None:
        dist.barrier()


# ----------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        self.samples, self.reasons, self._stop, self._thr = [], set(), threading.Event(), None
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self._nv = None

    def _run(self):
        nv = self._nv
        names = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                self.reasons.update(k for k, bit in names.items() if r & bit)
            except Exception:
                pass
            self._stop.wait(0.005)

    def __enter__(self):
        if self._nv:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr:
            self._thr.join()

    def summary(self):
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# -------------------------------------------------------------------------------------------- workloads
def make_workload(kind, rank, order=None):
    """The benchmarked workload of this rank: (Workload descriptor, number of templates per step)."""
    w, b = _make_workload(kind, rank)
    if order is not None:
        w.order = order   # order sweep
    return w, b


def _make_workload(kind, rank):
    from harness import inputs
    if kind == "year":
        w = inputs.config(2)
        if rank:  # other ranks: same shape, their own seeded source
            w.sources = [inputs.draw_gb(np.random.default_rng(2204 + rank))]
        return w, 1
    if kind == "batch":
        w = inputs.config(3)
        lo, hi = 0, len(w.sources)
        return w, hi - lo
    if kind == "tiny":
        return inputs.config(1), 1
    if kind == "4yr":
        return inputs.config(4), 1
    if kind in ("chirp", "hybrid"):   # hybrid: config 5 run (i), TDI-1 on equal-arm constant delays
        return inputs.config(5), 1
    raise ValueError(kind)


def gb_waveform_device(srcs, n, dt, t0, device):
    from harness import inputs
    return inputs.gb_waveform_device(srcs, n, dt, t0, device)


# ------------------------------------------------------------------------------------------ CPU oracle
def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def omp_threads():
    """Threads the oracle's OpenMP loops use in this process (it has no setter: OMP_NUM_THREADS or all cores)."""
    try:
        return max(1, int(os.environ.get("OMP_NUM_THREADS", "")))
    except ValueError:
        return os.cpu_count() or 1


def time_oracle(w, target_s=12.0):
    """The oracle as it stands (oracle/lr_oracle.cpp, fp64 arithmetic, OpenMP over samples) on a window of
    the workload's first template, sized for about target_s of host time.  Returns (samples/s, info)."""
    from oracle import oracle as orc
    tab = w.table()
    O = orc.Oracle(tab, w.dt, w.t0, w.order)
    hp, hc = w.waveform(0)
    s = w.sources[0]
    mp, mf, mb = O.margins(w.tdi_gen)
    ch = {"XYZ": 0, "AET": 1, "XYZ_AET": 2}[w.channels]
    mid = max(mf, w.n // 8)

    def run(m):
        lo, hi = mid, min(mid + m, w.n - mb)
        t0 = time.perf_counter()
        y = O.project(hp, hc, s.beta, s.lam, s.psi, lo=max(mp, lo - (mf - mp)), hi=hi, precision="d")
        O.tdi(y, w.tdi_gen, nested=True, channels=ch, lo=lo, hi=hi, precision="d")
        return time.perf_counter() - t0, hi - lo

    t_probe, m_probe = run(2000)
    m = int(max(2000, min(w.n - mb - mid, m_probe * target_s / max(t_probe, 1e-6))))
    t, m = run(m)
    return m / t, {"cores": omp_threads(), "kind": "oracle", "cpu_model": cpu_model(),
                   "sample": f"{m} consecutive samples starting at n/8 of template 0 (projection + TDI-{w.tdi_gen}, "
                             f"fp64 build of the oracle, OpenMP over samples), {t:.1f} s wall"}


def time_oracle_one_thread(args, target_s):
    """The same measurement in a child process with OMP_NUM_THREADS=1 (PAPER.md:273 quotes "a single ... CPU
    processor"): the oracle is not touched, the child is `bench.py --impl reference`."""
    env = dict(os.environ, OMP_NUM_THREADS="1")
    cmd = [sys.executable, os.path.abspath(__file__), "--impl", "reference", "--workload", args.workload, "--steps", "1",
           "--warmup", "0", "--cpu-seconds", str(target_s)]
    if args.order is not None:
        cmd += ["--order", str(args.order)]
    try:
        r = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=60 + 20 * target_s)
        line = [ln for ln in r.stdout.splitlines() if ln.startswith("{")][-1]
        d = json.loads(line)["cpu_baseline"]
        return {"value": d["value"], "unit": "samples/s", "cores": d["cores"], "sample": d["sample"]}
    except Exception as exc:   # never let the optional figure break the contract line
        return {"error": repr(exc)}


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores, same metric/config; rank 0 only.  Every step is a MEASURED
    bounded window of the workload (ms_per_step is the time of that window, `sample` says how long it was)."""
    if rank != 0:
        return
    w, _ = make_workload(args.workload, 0, args.order)
    vals, info = [], None
    per_step = min(args.cpu_seconds, max(1.0, min(20.0, 120.0 / max(1, args.steps + args.warmup))))
    t_steps = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        v, info = time_oracle(w, target_s=per_step)
        if i >= args.warmup:
            vals.append(v)
            t_steps.append(time.perf_counter() - t0)
    v = float(np.mean(vals))
    line = {"impl": "reference", "metric": "response samples/s (6-link proj + TDI-2, fp64)", "value": v,
            "unit": "samples/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * float(np.mean(t_steps)), "ms_per_whole_workload_extrapolated": 1e3 * w.n / v,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": workload_config(w, 1, args),
            "cpu_baseline": dict(info, value=v, unit="samples/s"),
            "e2e": {"value": v, "unit": "samples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def workload_config(w, batch, args):
    return {"workload": f"BASELINE.json configs[{ {'tiny': 0, 'year': 1, 'batch': 2, '4yr': 3, 'chirp': 4, 'hybrid': 4}[args.workload] }] ({w.name})",
            "batch": batch, "n": w.n, "dt": w.dt, "lagrange_order": w.order,
            "tdi_gen": 1 if args.workload == "hybrid" else w.tdi_gen,
            "chain": "nested", "channels": w.channels, "orbits": w.orbit_kind, "tdi_path": args.tdi_path,
            "y_precision": args.y_precision,
            "tdi_plan": "cached (built once per handle, like the paper's orbit arrays, PAPER.md:263; the `tdi_plan` key "
                        "has the step with the plan rebuilt in every call)",
            "l2": "flushed between steps (256 MiB memset outside the per-step event pairs)"}


def hbm_peak():
    """Measured HBM copy rate of this pool's B200 [GB/s] (driver-written MEASURED_PEAKS.json), else the fallback."""
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    except Exception:
        return 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md)"


def kernel_stats(ms_proj, ms_tdi, units, order, gen, nout, tdi_info, peak, hbm_gbs):
    """Per-kernel roofline figures.  units = template-samples one step processes.  frac_fp64: SURVEY §8(d)'s
    ALGORITHMIC instruction slots per second / measured FP64 issue rate; lr_tdi also gets frac_executed: the FMAs its
    FIR path really executes (3 channels x 4 series x taps x powers of tile time, from the handle) / the same rate;
    frac_hbm: algorithmic bytes per second / measured HBM copy rate.  `bound`: the larger of the two fractions."""
    T = order + 1
    path, taps, powers = tdi_info
    out = {}
    for name, ms, ops, nbytes in (("lr_project", ms_proj, ops_project(T), BYTES_PROJECT),
                                  ("lr_tdi", ms_tdi, ops_tdi(T, gen), bytes_tdi(nout))):
        rate = units / (ms * 1e-3)
        k = {"ms": ms, "alg_ops_per_sample": ops, "gops": ops * rate / 1e9, "frac_fp64": ops * rate / peak,
             "alg_bytes_per_sample": nbytes, "alg_GBps": nbytes * rate / 1e9, "frac_hbm": nbytes * rate / 1e9 / hbm_gbs}
        if name == "lr_tdi":
            k["path"] = path
            if path != "per_sample":
                ex = 3 * 4 * taps * powers
                k.update(executed_ops_per_sample=ex, fir_taps=taps, fir_powers=powers, frac_executed=ex * rate / peak,
                         executed_note="FMAs of the per-tile FIR filters (3 channels x 4 series x taps x powers of tile "
                                       "time); the algorithmic count charges a weight set per term and sample, so "
                                       "frac_fp64 > 1 here means fewer instructions, not a fuller pipe")
            else:
                k.update(executed_ops_per_sample=ops, frac_executed=ops * rate / peak)
        k["bound"] = "alu" if k.get("frac_executed", k["frac_fp64"]) >= k["frac_hbm"] else "hbm"
        out[name] = k
    return out


def timed_steps(lr, R, Rt, hp, hc, ang, y, out, reps, flush, stream):
    """reps x (lr_project, lr_tdi) on resident inputs; mean ms of each from CUDA events on the launch stream."""
    import torch
    ev = lambda: torch.cuda.Event(enable_timing=True)
    tp, tt = [], []
    for _ in range(reps):
        if flush is not None:
            flush.zero_()
        e0, e1, e2 = ev(), ev(), ev()
        e0.record(stream)
        R.project(hp, hc, *ang, y_out=y)
        e1.record(stream)
        Rt.tdi(y, out=out)
        e2.record(stream)
        e2.synchronize()
        tp.append(e0.elapsed_time(e1))
        tt.append(e1.elapsed_time(e2))
    return float(np.mean(tp)), float(np.mean(tt))


def batch_leg(lr, dev, local_rank, peak, hbm_gbs, reps=6):
    """BASELINE.json configs[2] (the MCMC batch) in the launch shape of `--workload batch`: ONE chunk of 64 of its
    1,024 templates at the full 1,576,800 samples, A,E,T: lr_project + lr_tdi per launch (the whole config is 16
    such launches), then parameters -> log L for the same 64 templates (lr_loglike_gb)."""
    import torch
    from harness import inputs
    w = inputs.config(3)
    nb, n = DEFAULT_CHUNK, w.n
    src = w.sources[:nb]
    R = lr.Response(w.table(), w.dt, w.order, w.tdi_gen, t0=w.t0, chain="nested", channels="AET")
    hp, hc = inputs.gb_waveform_device(src, n, w.dt, w.t0, dev)
    ang = ([s.beta for s in src], [s.lam for s in src], [s.psi for s in src])
    y = torch.empty((nb, 6, n), dtype=torch.float64, device=dev)
    out = torch.empty((nb, 3, n), dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream()
    clk = ClockSampler(local_rank)
    timed_steps(lr, R, R, hp, hc, ang, y, out, 2, None, stream)          # warm-up (builds the plan)
    l0 = lr.lr_launch_count()
    with clk:
        ms_p, ms_t = timed_steps(lr, R, R, hp, hc, ang, y, out, reps, None, stream)
        torch.cuda.synchronize()
    launches = lr.lr_launch_count() - l0
    ks = kernel_stats(ms_p, ms_t, float(nb) * n, w.order, w.tdi_gen, 3, R.tdi_info(), peak, hbm_gbs)
    dom = "lr_tdi" if ms_t >= ms_p else "lr_project"
    kd = ks[dom]
    leg = {"workload": "BASELINE.json configs[2] (MCMC batch): one launch of 64 of the 1,024 templates, 1,576,800 samples "
                       "each, Keplerian, order 25, nested TDI-2, A,E,T; inputs resident (8.8 GB per launch, far above L2)",
           "templates_per_launch": nb, "reps": reps, "ms_per_launch": ms_p + ms_t,
           "templates_per_s": nb / ((ms_p + ms_t) * 1e-3), "value": nb * n / ((ms_p + ms_t) * 1e-3), "unit": "samples/s",
           "gpu_launches": launches, "kernels": ks,
           "roofline": {"bound": "alu", "kernel": dom, "achieved": kd["gops"], "peak": peak / 1e9,
                        "unit": "Gop/s (FP64 thread-instruction slots, DFMA = 1)", "frac": kd["frac_fp64"],
                        "frac_executed": kd.get("frac_executed"),
                        "traffic": (ncu_counters("batch", dom)[0] or {}).get("dram_bytes"),
                        "traffic_source": "profiles/r2_ncu_counters.csv (workload batch)" if ncu_counters("batch", dom)[0]
                                          else ncu_counters("batch", dom)[1],
                        "path_frac": (ks["lr_project"]["alg_ops_per_sample"] + ks["lr_tdi"]["alg_ops_per_sample"]) * nb * n
                                     / ((ms_p + ms_t) * 1e-3) / peak},
           "clocks": clk.summary()}
    del y, hp, hc
    # parameters -> log L for the 64 templates (15 doubles in, 1 out per template; wall clock incl. the read-back)
    try:
        gb = np.array([[s.A * (1.0 + np.cos(s.iota) ** 2), -2.0 * s.A * np.cos(s.iota), s.f0, s.fdot, 0.0, s.phi0]
                       for s in src])
        m = lr.lr_fft_good_length(n)
        R.set_fft_length(m)
        nf = m // 2 + 1
        inv = torch.ones((3, nf), dtype=torch.float64, device=dev)
        inv[:, 0] = 0.0
        data_f = torch.fft.rfft(out[0], n=m, dim=-1).contiguous()
        del out
        tw = []
        for it in range(5):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            ll = R.loglike_gb(gb, *ang, n, data_f, inv, -2.0 * w.dt / m).cpu()
            if it >= 2:
                tw.append((time.perf_counter() - t0) * 1e3)
        leg["params_to_loglike"] = {"api": "lr_loglike_gb, 64 templates per call, transform zero padded to "
                                           f"{m} samples (LR_OPT_FFT_LENGTH)", "ms_per_call_wall": float(np.median(tw)),
                                    "loglike_per_s": nb / (float(np.median(tw)) * 1e-3),
                                    "h2d_bytes_per_call": nb * 15 * 8, "d2h_bytes_per_call": nb * 8,
                                    "log_l_of_the_data_template": float(ll[0])}
    except Exception as exc:
        leg["params_to_loglike"] = {"error": repr(exc)}
    return leg


def orders_leg(lr, dev, peak, hbm_gbs, orders=(1, 9, 25, 41), reps=5):
    """SURVEY §8(f) NEXT-3 (orders below 10 "can improve the speed", order 1 -> 25 changes the run
    time by "a factor of order unity"): the one-year shape at several Lagrange orders; per kernel the time and the
    fraction of the roof that binds at that order (FP64 issue or HBM)."""
    import torch
    from harness import inputs
    w = inputs.config(2)
    s = w.sources[0]
    hp_np, hc_np = w.waveform(0)
    hp, hc = torch.from_numpy(hp_np).to(dev)[None], torch.from_numpy(hc_np).to(dev)[None]
    ang = ([s.beta], [s.lam], [s.psi])
    y = torch.empty((1, 6, w.n), dtype=torch.float64, device=dev)
    out = torch.empty((1, 6, w.n), dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    rows = []
    for order in orders:
        R = lr.Response(w.table(), w.dt, order, 2, t0=w.t0, chain="nested", channels="XYZ_AET")
        timed_steps(lr, R, R, hp, hc, ang, y, out, 2, flush, stream)
        ms_p, ms_t = timed_steps(lr, R, R, hp, hc, ang, y, out, reps, flush, stream)
        ks = kernel_stats(ms_p, ms_t, float(w.n), order, 2, 6, R.tdi_info(), peak, hbm_gbs)
        row = {"order": order, "ms_per_step": ms_p + ms_t, "value": w.n / ((ms_p + ms_t) * 1e-3)}
        for name, k in ks.items():
            row[name] = {"ms": k["ms"], "bound": k["bound"], "frac": max(k["frac_fp64"], k["frac_hbm"]) if name == "lr_project"
                         else max(k["frac_executed"], k["frac_hbm"]), "frac_fp64": k["frac_fp64"], "frac_hbm": k["frac_hbm"],
                         **({"frac_executed": k["frac_executed"]} if name == "lr_tdi" else {})}
        rows.append(row)
        R.close()
    return {"workload": "BASELINE.json configs[1] shape (3,153,600 samples, X,Y,Z+A,E,T, plan cached) at other Lagrange orders",
            "frac_note": "per kernel: fraction of the roof that binds at that order; lr_project: algorithmic FP64 slots or "
                         "bytes; lr_tdi: executed FMAs of the FIR path or bytes",
            "orders": rows}


# --------------------------------------------------------------------------------------------- GPU arm
def run_gpu(args, rank, world, local_rank):
    import torch
    import paper_2204_06633_b200 as lr
    from paper_2204_06633_b200 import build as lrbuild
    lrbuild.ensure_built(local_rank)   # fresh checkout: compile the (git-ignored) library once
    lr.binding.lib()  # no CUDA extension -> fail loudly, there is no fallback
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    w, batch = make_workload(args.workload, rank, args.order)
    chunk = min(batch, args.chunk)
    n, T = w.n, w.order + 1
    nout = 6 if w.channels == "XYZ_AET" else 3
    R = lr.Response(w.table(), w.dt, w.order, w.tdi_gen, t0=w.t0, chain="nested", channels=w.channels,
                    tdi_path=args.tdi_path)
    R.set_y_precision(args.y_precision)
    Rt, tdi_gen = R, w.tdi_gen
    if args.workload == "hybrid":
        from harness import inputs as _inp
        eq = _inp.orbit_table("eq", w.t0, w.t0 + w.n * w.dt, const_ltt=_inp.ARM / _inp.C_LIGHT)
        tdi_gen = 1
        Rt = lr.Response(eq, w.dt, w.order, 1, t0=w.t0, chain="nested", channels=w.channels, tdi_path=args.tdi_path)
    stream = torch.cuda.current_stream()

    y = torch.empty((chunk, 6, n), dtype=torch.float64, device=dev)
    out = torch.empty((chunk, nout, n), dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    chunks = [(lo, min(lo + chunk, batch)) for lo in range(0, batch, chunk)]

    def angles(lo, hi):
        src = w.sources[lo:hi]
        return [s.beta for s in src], [s.lam for s in src], [s.psi for s in src]

    if batch == 1:
        hp_np, hc_np = w.waveform(0)
        h_cache = {0: (torch.from_numpy(hp_np).to(dev)[None], torch.from_numpy(hc_np).to(dev)[None])}
    else:
        h_cache = {}

    def chunk_inputs(lo, hi):
        if lo not in h_cache:
            h_cache.clear()
            h_cache[lo] = gb_waveform_device(w.sources[lo:hi], n, w.dt, w.t0, dev)
        return h_cache[lo]

    ev = lambda: torch.cuda.Event(enable_timing=True)

    def step(timed):
        """One pass over the whole batch; returns (ms project, ms tdi) from CUDA events on the launch stream."""
        tp = tt = 0.0
        for lo, hi in chunks:
            hp, hc = chunk_inputs(lo, hi)
            be, la, ps = angles(lo, hi)
            flush.zero_()
            e0, e1, e2 = ev(), ev(), ev()
            e0.record(stream)
            R.project(hp, hc, be, la, ps, y_out=y[:hi - lo])
            e1.record(stream)
            Rt.tdi(y[:hi - lo], out=out[:hi - lo])
            e2.record(stream)
            if timed:
                e2.synchronize()
                tp += e0.elapsed_time(e1)
                tt += e1.elapsed_time(e2)
        return tp, tt

    # (the roofline denominator is measured BEFORE the warm-up: the first step after its second-long DFMA kernel runs
    # 20 % slow, which would weigh on a run with few timed steps)
    peak = lr.lr_measure_fp64_peak(args.peak_seconds)   # FP64 thread-instructions / s, this device, now
    clk = ClockSampler(local_rank)     # (NVML is initialised here, not between the warm-up and the timed steps: 0.1 s
                                       # of idle GPU makes the next step 30 % slow)
    for _ in range(args.warmup):
        step(False)
    torch.cuda.synchronize()
    barrier()
    launches0 = lr.lr_launch_count()
    tps, tts = [], []
    wall0 = time.perf_counter()
    with clk:
        for _ in range(args.steps):
            a, b = step(True)
            tps.append(a)
            tts.append(b)
        torch.cuda.synchronize()
    barrier()
    wall = time.perf_counter() - wall0
    launches = lr.lr_launch_count() - launches0
    ms_proj, ms_tdi = float(np.mean(tps)), float(np.mean(tts))
    # lr_response: the same step as ONE call per chunk of templates, in time chunks through the small
    # y scratch of the handle (no [B,6,N] array)
    def step_response():
        t = 0.0
        for lo, hi in chunks:
            hp, hc = chunk_inputs(lo, hi)
            be, la, ps = angles(lo, hi)
            flush.zero_()
            e0, e1 = ev(), ev()
            e0.record(stream)
            R.response(hp, hc, be, la, ps, out=out[:hi - lo], tdi=Rt)
            e1.record(stream)
            e1.synchronize()
            t += e0.elapsed_time(e1)
        return t

    step_response()
    ms_resp = float(np.mean([step_response() for _ in range(max(2, min(args.steps, 20)))]))
    # likelihood stage: library rfft of the A,E,T (or last three) channels of one chunk +
    # lr_inner_product in LR_IP_DIFF mode against template 0 as the data
    lk = None
    try:
        nb = min(chunk, 8)
        ch3 = out[:nb, -3:, :].contiguous()
        nf = n // 2 + 1
        inv_psd = torch.ones((3, nf), dtype=torch.float64, device=dev)
        inv_psd[:, 0] = 0.0
        tf, ti = [], []
        for _ in range(5):
            e0, e1, e2 = ev(), ev(), ev()
            e0.record(stream)
            fh = (w.dt * torch.fft.rfft(ch3, dim=-1)).contiguous()
            e1.record(stream)
            lr.lr_inner_product(fh, fh[:1].contiguous(), inv_psd, -2.0 / (n * w.dt), mode=lr.LR_IP_DIFF)
            e2.record(stream)
            e2.synchronize()
            tf.append(e0.elapsed_time(e1))
            ti.append(e1.elapsed_time(e2))
        ms_ip = float(np.median(ti))
        hbm = None
        try:
            hbm = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))).get("hbm_gbs")
        except Exception:
            pass
        gbs = 40.0 * 3 * nf * nb / (ms_ip * 1e6)
        lk = {"templates": nb, "ms_rfft_library": float(np.median(tf)), "ms_lr_inner_product": ms_ip,
              "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm or 6650.0, "unit": "GB/s",
                           "frac": gbs / (hbm or 6650.0),
                           "peak_source": "MEASURED_PEAKS.json hbm_gbs (of measured)" if hbm else "fallback 6.65 TB/s",
                           "note": "algorithmic 40 B per bin and channel; > 1 when the spectra are still in L2"}}
        del fh, ch3, inv_psd
    except Exception as exc:   # never let the optional leg break the contract line
        lk = {"error": repr(exc)}
    # parameters -> log L in ONE call (waveform, projection, TDI, FFT and inner product on the device,
    # "only the scalar returns"): lr_loglike_gb on a 3-channel (A,E,T) handle of the same orbits.  Wall clock
    # around the call and the read-back of the scalars: host traffic is 120 B in and 8 B out per template.
    pl = None
    try:
        if args.workload not in ("year", "batch", "tiny") or not all(s.f0 > 0 for s in w.sources[:8]):
            raise RuntimeError("no Galactic-binary parameters in this workload")
        nb = min(chunk, 32)   # above 8 templates the call pipelines chunks of 8 (transforms beside the next response)
        Ra = lr.Response(w.table(), w.dt, w.order, w.tdi_gen, t0=w.t0, chain="nested", channels="AET")
        gb = np.array([[s.A * (1.0 + np.cos(s.iota) ** 2), -2.0 * s.A * np.cos(s.iota), s.f0, s.fdot, 0.0, s.phi0]
                       for s in w.sources[:nb]])
        be, la, ps = angles(0, nb)
        nf = n // 2 + 1
        inv_psd = torch.ones((3, nf), dtype=torch.float64, device=dev)
        inv_psd[:, 0] = 0.0
        aet0 = Ra.response_gb(gb[:1], be[:1], la[:1], ps[:1], n)
        data_f = torch.fft.rfft(aet0[0], dim=-1).contiguous()
        del aet0
        tw, td = [], []
        for it in range(7):
            torch.cuda.synchronize()
            t0w = time.perf_counter()
            e0, e1 = ev(), ev()
            e0.record(stream)
            ll = Ra.loglike_gb(gb, be, la, ps, n, data_f, inv_psd, -2.0 * w.dt / n)
            e1.record(stream)
            ll_h = ll.cpu()
            t1w = time.perf_counter()
            if it >= 2:
                tw.append((t1w - t0w) * 1e3)
                td.append(e0.elapsed_time(e1))
        ms_w, ms_d = float(np.median(tw)), float(np.median(td))
        pl = {"api": "lr_loglike_gb (host: 15 doubles in, 1 double out per template)", "templates": nb,
              "ms_per_call_wall": ms_w, "ms_per_call_device": ms_d, "ms_lr_response_gb": None,
              "value": nb * n / (ms_w * 1e-3), "unit": "samples/s", "loglike_per_s": nb / (ms_w * 1e-3),
              "h2d_bytes_per_call": int(nb * 15 * 8), "d2h_bytes_per_call": int(nb * 8),
              "log_l_of_the_data_template": float(ll_h[0])}
        outg = torch.empty((nb, 3, n), dtype=torch.float64, device=dev)
        tg = []
        for it in range(5):
            e0, e1 = ev(), ev()
            e0.record(stream)
            Ra.response_gb(gb, be, la, ps, n, out=outg)
            e1.record(stream)
            e1.synchronize()
            tg.append(e0.elapsed_time(e1))
        pl["ms_lr_response_gb"] = float(np.median(tg[1:]))
        # the same call with the transform zero padded to a length without large prime factors (LR_OPT_FFT_LENGTH)
        m = lr.lr_fft_good_length(n)
        if m != n:
            Ra.set_fft_length(m)
            mf_ = m // 2 + 1
            inv_m = torch.ones((3, mf_), dtype=torch.float64, device=dev)
            inv_m[:, 0] = 0.0
            aet0 = Ra.response_gb(gb[:1], be[:1], la[:1], ps[:1], n)
            data_m = torch.fft.rfft(aet0[0], n=m, dim=-1).contiguous()
            del aet0
            tw = []
            for it in range(7):
                torch.cuda.synchronize()
                t0w = time.perf_counter()
                ll_m = Ra.loglike_gb(gb, be, la, ps, n, data_m, inv_m, -2.0 * w.dt / m).cpu()
                t1w = time.perf_counter()
                if it >= 2:
                    tw.append((t1w - t0w) * 1e3)
            pl["padded_fft"] = {"n_fft": int(m), "ms_per_call_wall": float(np.median(tw)),
                                "loglike_per_s": nb / (float(np.median(tw)) * 1e-3),
                                "log_l_of_the_data_template": float(ll_m[0])}
            Ra.set_fft_length(0)
            del data_m, inv_m

        del outg, data_f, inv_psd, Ra
    except Exception as exc:   # never let the optional leg break the contract line
        pl = {"error": repr(exc)}
    if world > 1:   # the path's only exchange: all-gather of the scalars; every rank takes part
        if sum_over_ranks(0.0 if "error" in pl else 1.0) == world:
            full = lr.gather_scalars(ll, pl["templates"] * world, rank, world)
            torch.cuda.synchronize()
            pl["gathered_scalars"] = int(full.numel())
    # the same steps with the FIR plan rebuilt by every lr_tdi call (plan kernel inside the timed region)
    Rt.set_plan_cache(False)
    cold = [step(True) for _ in range(max(3, min(args.steps, 10)))]
    Rt.set_plan_cache(True)
    step(False)
    torch.cuda.synchronize()
    ms_tdi_cold = float(np.mean([b for _, b in cold]))
    ms_step = max_over_ranks(ms_proj + ms_tdi)
    units = sum_over_ranks(float(batch) * n)
    value = units / (ms_step * 1e-3)
    templates = sum_over_ranks(float(batch))

    # end to end through the C ABI with pinned HOST buffers (H2D + project + TDI + D2H inside the timed region)
    eb = min(batch, chunk if args.workload == "batch" else args.e2e_templates)   # batch: one whole launch chunk
    hp_h = torch.empty((eb, n), dtype=torch.float64).pin_memory()
    hc_h = torch.empty((eb, n), dtype=torch.float64).pin_memory()
    out_h = torch.empty((eb, nout, n), dtype=torch.float64).pin_memory()
    hp_d, hc_d = chunk_inputs(0, min(chunk, batch))
    hp_h.copy_(hp_d[:eb].cpu())
    hc_h.copy_(hc_d[:eb].cpu())
    be, la, ps = angles(0, eb)
    for _ in range(max(1, min(args.warmup, 3))):
        R.response_host(hp_h, hc_h, be, la, ps, out_h, tdi=Rt)
    torch.cuda.synchronize()
    barrier()
    e2e_ms = []
    for _ in range(max(3, min(args.steps, 10))):
        flush.zero_()
        torch.cuda.synchronize()
        e0, e1 = ev(), ev()
        e0.record(stream)
        R.response_host(hp_h, hc_h, be, la, ps, out_h, tdi=Rt)
        e1.record(stream)
        e1.synchronize()
        e2e_ms.append(e0.elapsed_time(e1))
    e2e_ms = max_over_ranks(float(np.mean(e2e_ms)))
    e2e_units = sum_over_ranks(float(eb) * n)

    if rank != 0:
        return
    hbm_gbs, hbm_src = hbm_peak()
    ks = kernel_stats(ms_proj, ms_tdi, float(batch) * n, w.order, tdi_gen, nout, Rt.tdi_info(), peak, hbm_gbs)
    dom = "lr_tdi" if ms_tdi >= ms_proj else "lr_project"
    kd = ks[dom]
    # ncu-only counters of the two kernels: from the tracked capture, valid only for the build it was taken on
    ncu = {}
    for api in ("lr_project", "lr_tdi"):
        c, why = ncu_counters(args.workload, api) if (args.order is None and args.tdi_path == "auto") else (None, "non-default order or TDI path")
        ncu[api] = c if c is not None else {"unavailable": why}
    traffic = ncu[dom].get("dram_bytes")
    line = {
        "metric": "response samples/s (6-link proj + TDI-2, fp64)" if args.workload != "batch"
                  else "response samples/s (6-link proj + TDI-2 AET, fp64), batched",
        "value": value, "unit": "samples/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": workload_config(w, batch, args),     # (the same object in the --impl reference arm)
        "launch": {"chunk_templates": chunk, "parallelism": f"{world} rank(s), templates sharded, no collective"},
        "templates_per_s": templates / (ms_step * 1e-3),
        "e2e": {"value": e2e_units / (e2e_ms * 1e-3), "unit": "samples/s", "ms_per_step": e2e_ms,
                "templates": eb, "h2d_bytes_per_step": 2 * eb * n * 8, "d2h_bytes_per_step": nout * eb * n * 8,
                "api": "lr_response_host (pinned host buffers)"},
        "gpu_launches": launches,
        "kernels": ks,
        "likelihood": lk,
        "params_to_loglike": pl,
        "lr_response": {"ms_per_step": ms_resp, "note": "one call, h -> out, y only in a scratch of two <= 1 GB slots"},
        "tdi_plan": {"cached_between_calls": True, "ms_tdi_with_plan_rebuilt_every_call": ms_tdi_cold,
                     "value_with_plan_rebuilt_every_call": units / (max_over_ranks(ms_proj + ms_tdi_cold) * 1e-3)
                     if world == 1 else None},
        "roofline": {"bound": "alu", "kernel": dom + (" (tdi_fir_apply_kernel)" if dom == "lr_tdi" and ks["lr_tdi"]["path"] != "per_sample" else ""),
                     "achieved": kd["gops"], "peak": peak / 1e9,
                     "unit": "Gop/s (FP64 thread-instruction slots, DFMA = 1)", "frac": kd["frac_fp64"],
                     "frac_executed": kd.get("frac_executed"),
                     "traffic": traffic,
                     "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum per launch, profiles/r2_ncu_counters.csv"
                                       if traffic is not None else ncu[dom].get("unavailable"),
                     "peak_source": f"lr_measure_fp64_peak({args.peak_seconds} s DFMA kernel) on this device, this run",
                     "peak_nominal": torch.cuda.get_device_properties(dev).multi_processor_count * 64 *
                                     (clk.max_mhz or 1965) * 1e-3,   # SMs x 64 FP64 lanes x max SM clock [Gop/s]
                     "hbm_peak_GBps": hbm_gbs, "hbm_peak_source": hbm_src,
                     "ncu": ncu, "csrc_sha256": csrc_hash(),
                     "path_frac": (ks["lr_project"]["alg_ops_per_sample"] + ks["lr_tdi"]["alg_ops_per_sample"]) * batch * n
                                  / ((ms_proj + ms_tdi) * 1e-3) / peak},
        "clocks": clk.summary(), "wall_s_timed_region": wall,
    }
    # free the main workload's buffers before the extra legs
    del y, out, flush, hp_h, hc_h, out_h
    h_cache.clear()
    torch.cuda.empty_cache()
    if world == 1 and args.workload == "year" and args.order is None and args.tdi_path == "auto":
        if not args.no_batch_leg:
            try:
                line["batch"] = batch_leg(lr, dev, local_rank, peak, hbm_gbs)
            except Exception as exc:   # never let an extra leg break the contract line
                line["batch"] = {"error": repr(exc)}
            torch.cuda.empty_cache()
        if not args.no_orders_leg:
            try:
                line["orders"] = orders_leg(lr, dev, peak, hbm_gbs)
            except Exception as exc:
                line["orders"] = {"error": repr(exc)}
    if world == 1 and not args.no_cpu_baseline:
        v, info = time_oracle(w, target_s=args.cpu_seconds)
        line["cpu_baseline"] = dict(info, value=v, unit="samples/s",
                                    one_thread=time_oracle_one_thread(args, args.cpu_seconds))
    print(json.dumps(line), flush=True)


def run_gpu_time_sharded(args, rank, world, local_rank):
    """N > 1, one template split along time: every rank holds its span of h plus the halo and computes its span
    of out with lr_response_span; no collective on the data path.  Strong scaling: value = n / max-over-ranks time."""
    import torch
    import paper_2204_06633_b200 as lr
    from paper_2204_06633_b200 import build as lrbuild
    lrbuild.ensure_built(local_rank)
    lr.binding.lib()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    w, batch = make_workload(args.workload, 0, args.order)
    if batch != 1:
        raise SystemExit("--shard time needs a single-template workload")
    s = w.sources[0]
    R = lr.Response(w.table(), w.dt, w.order, w.tdi_gen, t0=w.t0, chain="nested", channels=w.channels,
                    tdi_path=args.tdi_path)
    lo, hi, unit = R.span_halo()
    first, count, h_first, h_len = lr.shard_time(w.n, rank, world, unit, lo, hi)
    hp, hc = w.waveform(0)
    hps = torch.from_numpy(hp[h_first:h_first + h_len].copy()).to(dev)[None]
    hcs = torch.from_numpy(hc[h_first:h_first + h_len].copy()).to(dev)[None]
    out = torch.empty((1, R.n_out, max(count, 1)), dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    def step():
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        if count:
            R.response_span(hps, hcs, h_first, [s.beta], [s.lam], [s.psi], w.n, first, count, out=out[:, :, :count])
        e1.record(stream)
        e1.synchronize()
        return e0.elapsed_time(e1)

    peak = lr.lr_measure_fp64_peak(args.peak_seconds)
    clk = ClockSampler(local_rank)
    for _ in range(args.warmup):
        step()
    barrier()
    torch.cuda.synchronize()
    launches0 = lr.lr_launch_count()
    with clk:
        ms = [step() for _ in range(args.steps)]
        torch.cuda.synchronize()
    barrier()
    launches = lr.lr_launch_count() - launches0
    ms_step = max_over_ranks(float(np.mean(ms)))
    if rank != 0:
        return
    T = w.order + 1
    ach = (ops_tdi(T, w.tdi_gen) + ops_project(T)) * w.n / (ms_step * 1e-3)
    print(json.dumps({
        "metric": "response samples/s (6-link proj + TDI-2, fp64)", "value": w.n / (ms_step * 1e-3),
        "unit": "samples/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step,
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": dict(workload_config(w, 1, args), parallelism=f"{world} ranks, one template split along time "
                       "(lr_response_span, halos recomputed, no collective)"),
        "gpu_launches": launches, "e2e": None,
        "roofline": {"bound": "alu", "kernel": "whole path (lr_response_span)", "achieved": ach / 1e9,
                     "peak": world * peak / 1e9, "unit": "Gop/s (FP64 thread-instruction slots, DFMA = 1)",
                     "frac": ach / (world * peak), "traffic": None,
                     "peak_source": "lr_measure_fp64_peak on rank 0 x ranks"},
        "clocks": clk.summary()}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="year", choices=["year", "batch", "tiny", "4yr", "chirp", "hybrid"])
    ap.add_argument("--order", type=int, default=None, help="override the Lagrange order (order sweep)")
    ap.add_argument("--chunk", type=int, default=DEFAULT_CHUNK, help="templates per launch (batch workload)")
    ap.add_argument("--e2e-templates", type=int, default=4)
    ap.add_argument("--peak-seconds", type=float, default=1.0)
    ap.add_argument("--cpu-seconds", type=float, default=10.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--y-precision", default="extended", choices=["extended", "plain"],
                    help="LR_OPT_Y_PRECISION of lr_project (the library's default is extended)")
    ap.add_argument("--no-batch-leg", action="store_true", help="skip the 64-template launch of configs[2]")
    ap.add_argument("--no-orders-leg", action="store_true", help="skip the Lagrange-order sweep")
    ap.add_argument("--tdi-path", default="auto", choices=["auto", "per_sample", "fir3", "fir4"])
    ap.add_argument("--shard", default="templates", choices=["templates", "time"],
                    help="N > 1: 'templates' = every rank its own template(s) (weak scaling, default); 'time' = ONE "
                         "template split along time with lr_response_span (strong scaling, 'year'/'4yr'/'chirp')")
    ap.add_argument("--ncu-import", default=None, help="raw-page CSV of an ncu full capture: refresh profiles/r2_ncu_counters.csv (no GPU needed)")
    ap.add_argument("--ncu-workload", default="year", help="workload label of --ncu-import rows: year | batch")
    args = ap.parse_args()
    if args.ncu_import:
        ncu_import(args.ncu_import, args.ncu_workload)
        return
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if world > 1:
        import torch
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    try:
        if args.shard == "time":
            run_gpu_time_sharded(args, rank, world, local_rank)
        else:
            run_gpu(args, rank, world, local_rank)
    finally:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
