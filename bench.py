#!/usr/bin/env python
"""bench.py -- throughput of the determinant-form Wick contraction hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg3]

A "step" is one pass of the whole hot path (steps a3-a6 of DESIGN.md: propagator staging, unique minor
determinants, weighted products, momentum projection) over one batch of synthetic input: the FULL term
list of the workload on `timeslices_per_step` (default 4, contiguous) full timeslices of its lattice per GPU.
Default workload: cfg3 (Helium-4, L = 32, 2716 x 2716 terms, 858,050 unique 6x6 minors per site), the
configuration BASELINE.json's target is quoted on.  Metric: correlator timeslices/s (whole job).  The timed loop
runs with the library's per-launch events OFF; the kernel classes are timed in a separate pass.  The same JSON
line carries the rooflines of the minors kernels (FP64 ALU: flops the kernels EXECUTE / time / the DFMA rate
measured in this run) and of the reduction (HBM), and a "workloads" object with the Lithium-7-sized
configurations (cfg4, cfg4b), measured the same way in this run.

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (oracle/, as it stands) on a
bounded sample of the same workload instead.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from wick_inputs import CONFIGS, make_propagators_numpy, make_random_term_list  # noqa: E402

# Algorithmic flops: FMA = 2 flops, complex FMA = 8, complex mul = 6.
def flops_lu(n: int) -> float:
    if n <= 1:
        return 0.0
    if n == 2:
        return 14.0
    if n == 3:
        return 64.0
    if n == 4:
        return 220.0
    return 8.0 * (n - 1) * n * (2 * n - 1) / 6 + 6.0 * n * (n - 1) / 2 + 15.0 * (n - 1) + 3.0 * (n * (n + 1) / 2 - 1)

def executed_flops_per_site(n: int, row_in_order: np.ndarray, cols_in_order: np.ndarray, grid_cols=None) -> float:
    """Flops the minors kernel actually executes per site for one flavour, from the order in which it
    walks the minors (Terms.minor_order): the pivoted-LU state is kept across consecutive minors that share the row
    tuple and leading columns, so the K = n-4 pivot steps run once per (row tuple, first K columns), the 2x2 / 3x3
    minors of the Schur complement once per (.., first K+2 / K+3 columns), and only the last column once per minor."""
    nm = len(row_in_order)
    if n <= 2 or nm == 0:
        return nm * flops_lu(n)
    c = cols_in_order.astype(np.int64)
    same_row = row_in_order[1:] == row_in_order[:-1]

    def same_lead(k):
        return same_row & np.all(c[1:, :k] == c[:-1, :k], axis=1)
    if n == 3:                                                     # cofactors of the last column per (rows, b0, b1)
        return (1 + int(np.count_nonzero(~same_lead(2)))) * 42.0 + nm * 22.0
    K = n - 4
    if grid_cols is not None:
        # minors_reg_kernel (grid tables, n = 6): per (row tuple, K leading columns) instance the pivot steps and one Schur
        # column per candidate column index; per (i2, i3) pair node 4 complex multiplications by the pivot product and six
        # 2x2 minors; per (i2, i3, i4) node four signed 3x3 minors; per minor a 4-term Laplace sum
        f_col_ = 8.0 * sum(n - 1 - i for i in range(K))
        f_start_ = sum(8.0 * sum(n - 1 - i for i in range(J)) + (n - J) + 14.0 + 6.0 * (n - 1 - J) + (6.0 if J else 0.0)
                       for J in range(K))
        cc = [tuple(int(x) for x in t) for t in grid_cols]
        inst, pairs, thirds = {}, set(), set()
        for t in cc:
            inst.setdefault(t[:K], set()).update(t[K:])
            pairs.add(t[:K + 2])
            thirds.add(t[:K + 3])
        per_row = (len(inst) * f_start_ + sum(len(v) for v in inst.values()) * f_col_ + len(pairs) * (84.0 + 24.0)
                   + len(thirds) * 88.0 + len(cc) * 30.0)
        return per_row * (nm // len(cc))
    f_col = 8.0 * sum(n - 1 - i for i in range(K))
    f_start = sum(8.0 * sum(n - 1 - i for i in range(J)) + (n - J) + 14.0 + 6.0 * (n - 1 - J) + (6.0 if J else 0.0)
                  for J in range(K))
    f_pair, f_third, f_finish = 2 * f_col + 84.0, f_col + 88.0, f_col + 36.0
    if n == 6:
        # minors6_cached_kernel: every Schur column of a (row tuple, b0, b1) instance is computed once, right after the two
        # pivot steps (column indices max(b1 + 1, 3) .. 11, plus index 2 for b1 < 2); the levels only combine cached columns
        first = np.concatenate(([True], ~same_lead(K)))
        b1 = c[first, 1]
        n_cols = int(np.sum(12 - np.maximum(b1 + 1, 3) + (b1 < 2)))
        n_pair = 1 + int(np.count_nonzero(~same_lead(K + 2)))
        n_third = 1 + int(np.count_nonzero(~same_lead(K + 3)))
        return int(first.sum()) * f_start + n_cols * f_col + n_pair * 84.0 + n_third * 88.0 + nm * 36.0
    if n in (10, 11):
        # minors_large_cached_kernel: the 12 - K Schur columns of a (row tuple, leading columns) instance are computed once
        n_inst = 1 + int(np.count_nonzero(~same_lead(K)))
        n_pair = 1 + int(np.count_nonzero(~same_lead(K + 2)))
        n_third = 1 + int(np.count_nonzero(~same_lead(K + 3)))
        return n_inst * (f_start + (12 - K) * f_col) + n_pair * 84.0 + n_third * 88.0 + nm * 36.0
    n_fresh = 1 + int(np.count_nonzero(~same_lead(K)))
    n_pair = 1 + int(np.count_nonzero(~same_lead(K + 2)))
    n_third = 1 + int(np.count_nonzero(~same_lead(K + 3)))
    return n_fresh * f_start + n_pair * f_pair + n_third * f_third + nm * f_finish


FLOPS_PER_TERM = 14.0
FP64_PEAK_DERIVED_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12     # 148 SMs x 64 DFMA lanes x 2 flop x 1.965 GHz = 37.2


def read_measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return {}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu, self.rows, self.proc = gpu_index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.gpu)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm = [float(r[1]) for r in self.rows if len(r) >= 9 and r[1].replace(".", "").isdigit()]
        mx = [float(r[2]) for r in self.rows if len(r) >= 9 and r[2].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[k] for r in self.rows if len(r) >= 9 for k in range(4) if r[5 + k] == "Active"})
        pw = [float(r[3]) for r in self.rows if len(r) >= 9 and r[3].replace(".", "").isdigit()]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "reasons": reasons, "samples": len(sm)}


def workload_terms(wk, cfg):
    if cfg.random_list:
        return wk.build_terms_from_list(*make_random_term_list(cfg.seed, cfg.n_u, cfg.n_d, cfg.n_random_terms))
    return wk.build_terms(cfg.nucleus)


def _oracle_site_runner(cfg, method: str):
    """Closure that evaluates one site of the workload with the oracle.  method 'A' = two fresh determinants per term
    (the paper's vanilla method: the oracle proper); 'B' = every distinct minor once per site, then the
    term sum (the paper's improved method: what its SERIAL C / OPENMP C rows run)."""
    from oracle import wick_oracle as wo
    U, D = make_propagators_numpy(cfg.seed, cfg.L, cfg.T, t0=0, nt=1)
    if cfg.random_list:
        lst = make_random_term_list(cfg.seed, cfg.n_u, cfg.n_d, cfg.n_random_terms)
        return lambda s: wo.site_terms_value(U[0, s], D[0, s], *lst)
    sink = wo.merged_terms(cfg.nucleus)
    if method == "B":
        return lambda s: wo.site_value_method_b(U[0, s], D[0, s], sink)
    return lambda s: wo.site_value_outer(U[0, s], D[0, s], sink)


def _oracle_worker(args):
    name, method, sites = args
    os.environ["OMP_NUM_THREADS"] = "1"
    run = _oracle_site_runner(CONFIGS[name], method)
    t0 = time.perf_counter()
    for s in sites:
        run(s)
    return time.perf_counter() - t0


def oracle_seconds_per_site(cfg, n_sites: int, method: str = "A"):
    """Time the oracle on n_sites sites of the workload, one core.  Returns (seconds per site, threads used)."""
    run = _oracle_site_runner(cfg, method)
    t0 = time.perf_counter()
    for s in range(n_sites):
        run(s)
    return (time.perf_counter() - t0) / n_sites, 1          # numpy elementwise code: one thread


def oracle_sites_per_second_all_cores(cfg, key: str, sites_per_worker: int, method: str = "A"):
    """The same oracle code on every host core: one process per core, each evaluating its own sites (sites are
    independent, Eq. A5).  Returns (sites per second of the whole pool, processes used)."""
    import multiprocessing as mp
    cores = len(os.sched_getaffinity(0))
    jobs = [(key, method, list(range(w * sites_per_worker, (w + 1) * sites_per_worker))) for w in range(cores)]
    with mp.get_context("spawn").Pool(cores) as pool:
        t0 = time.perf_counter()
        busy = pool.map(_oracle_worker, jobs)
        wall = time.perf_counter() - t0
    # the pool start-up (interpreter + numpy import + term expansion per process) is not oracle work: use the slowest worker
    return cores * sites_per_worker / max(max(busy), 1e-9), cores, wall


def cpu_baseline_rows(cfg, key: str, sites_a: int, all_cores: bool):
    """cpu_baseline of the bench line: the oracle as it stands (method A) on one core, plus the same
    on all host cores and the plain method-B CPU row, each on a bounded sample scaled by L^3 sites per timeslice."""
    sps, cores = oracle_seconds_per_site(cfg, sites_a)
    out = {"value": 1.0 / (sps * cfg.volume), "unit": "timeslices/s", "cores": cores, "kind": "oracle",
           "sample": f"{sites_a} site(s) of {cfg.name} (full term list), {sps:.3g} s per site, scaled by L^3 = {cfg.volume} sites per timeslice",
           "host_cores_available": len(os.sched_getaffinity(0))}
    if not cfg.random_list:
        n_b = max(sites_a, 2)
        sps_b, _ = oracle_seconds_per_site(cfg, n_b, "B")
        out["method_b_one_core"] = {"value": 1.0 / (sps_b * cfg.volume), "unit": "timeslices/s", "cores": 1, "kind": "oracle (method B: unique minors once per site, PAPER.md:294)",
                                    "sample": f"{n_b} sites, {sps_b:.3g} s per site"}
    if all_cores:
        try:
            rate, n_proc, wall = oracle_sites_per_second_all_cores(cfg, key, 1, "A")
            out["all_cores"] = {"value": rate / cfg.volume, "unit": "timeslices/s", "cores": n_proc, "kind": "oracle",
                                "sample": f"1 site per process, {n_proc} processes, slowest worker as the time (pool wall {wall:.1f} s)"}
            if not cfg.random_list:
                rate_b, n_proc, wall = oracle_sites_per_second_all_cores(cfg, key, 2, "B")
                out["method_b_all_cores"] = {"value": rate_b / cfg.volume, "unit": "timeslices/s", "cores": n_proc,
                                             "kind": "oracle (method B)", "sample": f"2 sites per process, {n_proc} processes"}
        except Exception as exc:                                   # a missing /dev/shm or fork limit must not kill the bench line
            out["all_cores"] = {"unavailable": repr(exc)}
    return out


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores; each step = `sites` sites of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    sites = args.ref_sites
    for _ in range(args.warmup):
        oracle_seconds_per_site(cfg, 1)
    t0 = time.perf_counter()
    per_site = []
    for _ in range(args.steps):
        sps, cores = oracle_seconds_per_site(cfg, sites)
        per_site.append(sps)
    wall = time.perf_counter() - t0
    sps = float(np.mean(per_site))
    value = 1.0 / (sps * cfg.volume)                         # timeslices/s
    line = {
        "impl": "reference", "metric": "correlator_timeslices_per_s", "value": value, "unit": "timeslices/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": wall / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64 (complex128)", "data": "synthetic",
        "config": {"workload": cfg.name, "L": cfg.L, "T": cfg.T, "n_u": cfg.n_u, "n_d": cfg.n_d},
        "cpu_baseline": {"value": value, "unit": "timeslices/s", "cores": cores, "kind": "oracle",
                         "sample": f"{sites} site(s) of {cfg.name} per step, scaled by L^3 = {cfg.volume} sites per timeslice"},
        "e2e": {"value": value, "unit": "timeslices/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def kernel_source_hash() -> str:
    """sha256 over the CUDA sources: keys the committed ncu traffic figures to the kernels they were measured on."""
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_2411_08962_b200", "csrc")
    for name in sorted(os.listdir(csrc)):
        if name.endswith((".cu", ".cuh", ".h", ".cpp")):
            with open(os.path.join(csrc, name), "rb") as f:
                h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()[:16]


def read_traffic(cfg_name: str):
    """DRAM bytes per launch from the committed `ncu --set full` capture (profiles/r02_roofline_traffic.json.txt), only
    if that capture was taken on the kernel sources of this tree; otherwise null with the reason."""
    path = os.path.join(ROOT, "profiles", "r02_roofline_traffic.json.txt")
    try:
        with open(path) as f:
            rec = json.load(f)
    except Exception:
        return None, "no committed capture (profiles/r02_roofline_traffic.json.txt)"
    here = kernel_source_hash()
    if rec.get("kernel_source_hash") != here:
        return None, f"stale: capture taken on kernel sources {rec.get('kernel_source_hash')}, this tree is {here}"
    return rec.get("workloads", {}).get(cfg_name), f"profiles/r02_roofline_traffic.json.txt ({rec.get('command', 'ncu --set full')})"


def minors_kernel_names(info, outer: bool):
    def one(n):
        if n == 6 and outer:
            return "minors_reg_kernel<6,10>"
        return {6: "minors6_cached_kernel", 10: "minors_large_cached_kernel<10>", 11: "minors_large_cached_kernel<11>"}.get(n, f"minors_kernel<{n}>")
    return " / ".join(one(n) for n in (info.n_u, info.n_d))


def reduce_executed_flops_per_site(terms, info) -> float:
    """Flops the weighted-product kernel executes per site.  Factorised lists (reduce_staged_kernel): Q = B . MU row
    (2 DFMA per real coefficient and (u row tuple, source entry)), P likewise over the sink entries, one complex FMA per
    (u row tuple, d column tuple).  Flat lists: two complex multiplications and one addition per term."""
    if not info.is_outer_product:
        return float(info.n_terms) * FLOPS_PER_TERM
    sru, srd, sc, qcu, qcd, qc = terms.factors()
    real = bool(np.all(sc.imag == 0) and np.all(qc.imag == 0))
    per_entry = 4.0 if real else 8.0
    return per_entry * (info.n_source * info.n_rows_u + info.n_sink * info.n_cols_d) + 8.0 * info.n_rows_u * info.n_cols_d


def class_times(wk, torch, step, n_prof):
    """Per-class device time per step (CUDA events around every launch of a class, on the launching stream)."""
    wk.profile_enable(True)
    for _ in range(n_prof):
        step()
    torch.cuda.synchronize()
    prof = wk.profile_read()
    wk.profile_enable(False)
    return {k: (v[0] / n_prof, v[1] // n_prof) for k, v in prof.items()}


def rooflines(wk, cfg, terms, info, prof, ms_step, Tb, fp64_probe, hbm_gbs, d_runs):
    """roofline blocks of one workload: the minors kernels (FP64 ALU) and the weighted-product kernel (HBM)."""
    st_per_step = Tb * cfg.volume
    ms_minors = prof["minors_u"][0] + prof["minors_d"][0]
    ms_reduce, ms_project = prof["reduce"][0], prof["project"][0]
    n_minor_launches = prof["minors_u"][1] + prof["minors_d"][1]
    ur, uc, dr, dc = terms.tuples()
    mu_row, _, md_row, _ = terms.minors()
    ou, od = terms.minor_order(0), terms.minor_order(1)
    outer = bool(info.is_outer_product)
    exec_site = (executed_flops_per_site(info.n_u, mu_row[ou[0]], ou[1], uc if (outer and info.n_u == 6) else None),
                 executed_flops_per_site(info.n_d, md_row[od[0]], od[1], dc if (outer and info.n_d == 6) else None))
    exec_flop = st_per_step * (exec_site[0] + d_runs * exec_site[1])
    alg_flop = st_per_step * (info.n_minors_u * flops_lu(info.n_u) + d_runs * info.n_minors_d * flops_lu(info.n_d))
    executed_tf = exec_flop / (ms_minors * 1e-3) / 1e12 if ms_minors > 0 else 0.0
    peak = fp64_probe if fp64_probe else FP64_PEAK_DERIVED_TFLOPS
    traffic, traffic_src = read_traffic(cfg.name)
    minors = {
        "bound": "alu", "kernel": minors_kernel_names(info, outer) + " (a4, LU with partial pivoting)",
        "achieved": executed_tf, "peak": peak, "unit": "TFLOP/s", "frac": executed_tf / peak,
        "achieved_is": "flops the kernels execute (pivot steps and Schur columns shared by minors with equal row tuple and "
                       "leading columns, DESIGN.md 6b), counted on the host from the tables, / CUDA-event time of the minors launches",
        "peak_source": "register-only DFMA stream measured in this run (wick_measure_fp64_peak); MEASURED_PEAKS.json has no FP64 entry",
        "peak_spec_arithmetic": FP64_PEAK_DERIVED_TFLOPS, "frac_of_spec_arithmetic": executed_tf / FP64_PEAK_DERIVED_TFLOPS,
        "executed_flops_per_minor": {"u": exec_site[0] / max(info.n_minors_u, 1), "d": exec_site[1] / max(info.n_minors_d, 1)},
        "algorithmic_equivalent": {"tflops": alg_flop / (ms_minors * 1e-3) / 1e12 if ms_minors > 0 else None,
                                   "flops_per_minor": {"u": flops_lu(info.n_u), "d": flops_lu(info.n_d)},
                                   "note": "one full LU per unique minor (SURVEY 8d convention); not a roofline fraction"},
        "traffic": (traffic or {}).get("minors_dram_bytes_per_launch"), "traffic_source": traffic_src,
        "launches_per_step": int(n_minor_launches), "avg_launch_ms": ms_minors / max(n_minor_launches, 1),
        "kernel_share_of_step": ms_minors / ms_step,
        "per_flavour_ms_per_step": {"u": prof["minors_u"][0], "d": prof["minors_d"][0]},
    }
    red_flop = st_per_step * reduce_executed_flops_per_site(terms, info)
    red_bytes = st_per_step * 16.0 * (info.n_minors_u + info.n_minors_d * d_runs + 1)   # every minor read once + sigma
    reduce = {
        "bound": "hbm", "kernel": "reduce_staged_kernel (a5)" if outer else "reduce_flat_kernel (a5)",
        "achieved": red_bytes / (ms_reduce * 1e-3) / 1e9 if ms_reduce > 0 else None, "peak": hbm_gbs, "unit": "GB/s",
        "frac": (red_bytes / (ms_reduce * 1e-3) / 1e9 / hbm_gbs) if (ms_reduce > 0 and hbm_gbs) else None,
        "achieved_is": "16 B x unique minors x site-times (each minor read once) / CUDA-event time of the reduction launches",
        "peak_source": "MEASURED_PEAKS.json hbm_gbs" if hbm_gbs else "unavailable",
        "executed_tflops": red_flop / (ms_reduce * 1e-3) / 1e12 if ms_reduce > 0 else None,
        "executed_frac_of_fp64_peak": (red_flop / (ms_reduce * 1e-3) / 1e12 / peak) if ms_reduce > 0 else None,
        "traffic": (traffic or {}).get("reduce_dram_bytes_per_launch"), "traffic_source": traffic_src,
        "launches_per_step": int(prof["reduce"][1]), "avg_launch_ms": ms_reduce / max(prof["reduce"][1], 1),
        "kernel_share_of_step": ms_reduce / ms_step,
    }
    dram_step = (traffic or {}).get("dram_bytes_per_timeslice")
    return minors, reduce, {"project_ms_per_step": ms_project,
                            "dram_bytes_per_timeslice": dram_step,
                            "dram_over_algorithmic": (dram_step / (4608.0 * cfg.volume)) if dram_step else None,
                            "algorithmic_bytes_per_timeslice": 4608.0 * cfg.volume}


def bench_gevp(wk, torch, dev, Tb, steps, warmup):
    """Correlation matrix (GEVP, Sec. V) of two deuteron interpolators -- the p n product operator of cfg1 and
    the paper's Eq. (20) -- on the cfg1 lattice: wick_contract_many (every determinant once for the four entries) against four
    separate wick_contract calls on the same four term lists."""
    from wick_inputs import make_propagators_torch
    cfg = CONFIGS["cfg1"]
    ops = [wk.operator_from_nucleons(cfg.nucleus), wk.operator_paper(wk.OP_DEUTERON_EQ20)]
    m = wk.build_terms_matrix(ops)
    lists = [m[k][kp] for k in range(2) for kp in range(2)]
    U, D = make_propagators_torch(cfg.seed, cfg.L, cfg.T, dev, t0=0, nt=Tb)

    def many():
        return wk.contract_many(U, D, lists, cfg.momenta, cfg.L, Tb)

    def separate():
        return [wk.contract(U, D, t, cfg.momenta, cfg.L, Tb) for t in lists]

    out = {}
    for name, fn in (("contract_many", many), ("four_contract_calls", separate)):
        for _ in range(max(warmup, 3)):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        out[name] = e0.elapsed_time(e1) / steps
    Cm, Cs = many(), separate()
    same = all(bool(torch.allclose(Cm[e], Cs[e], rtol=1e-12, atol=0.0)) for e in range(4))
    i = lists[0].info
    return {"workload": "cfg1 lattice, 2 x 2 correlation matrix of {p0 n0 product, Eq. (20)}", "operators_terms": [o.n_terms for o in ops],
            "unique_minors_per_site": int(i.n_minors_u + i.n_minors_d), "terms_per_entry": [int(t.info.n_terms) for t in lists],
            "timeslices_per_step": Tb, "steps": steps, "ms_per_step": out["contract_many"], "value": Tb / (out["contract_many"] * 1e-3),
            "unit": "correlation-matrix timeslices/s", "ms_per_step_four_separate_calls": out["four_contract_calls"],
            "speedup_from_sharing_the_minors": out["four_contract_calls"] / out["contract_many"], "entries_agree_with_separate_calls": same}


def bench_workload(wk, torch, cfg, key, Tb, steps, warmup, dev, fp64_probe, hbm_gbs, isospin=False, sampler=None, flags=0):
    """One workload on this rank's GPU, device-resident inputs: timeslices/s, rooflines, launches.  Single-GPU path.
    isospin: one propagator for both flavours and the swap-symmetrised factorised list (WICK_BUILD_ISOSPIN)."""
    from wick_inputs import make_propagators_torch
    terms = wk.build_terms(cfg.nucleus, flags=wk.BUILD_ISOSPIN) if isospin else workload_terms(wk, cfg)
    info = terms.info
    n_mom = len(cfg.momenta)
    Tb = min(Tb, cfg.T)
    U, D = make_propagators_torch(cfg.seed, cfg.L, cfg.T, dev, t0=0, nt=Tb)
    if isospin:
        D = U
    ws = torch.empty(wk.contract_workspace_bytes(terms, cfg.L, Tb, n_mom), dtype=torch.uint8, device=dev)
    Cout = torch.empty((n_mom, Tb), dtype=torch.complex128, device=dev)

    def step():
        wk.contract(U, D, terms, cfg.momenta, cfg.L, Tb, workspace=ws, out=Cout, flags=flags)

    for _ in range(max(warmup, 3)):
        step()
    torch.cuda.synchronize()
    if sampler is not None:
        sampler.start()
    wk.launch_count(reset=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    ms_step = e0.elapsed_time(e1) / steps
    launches = wk.launch_count(reset=True)
    clocks = sampler.stop() if sampler is not None else None
    prof = class_times(wk, torch, step, max(1, min(3, steps)))
    wk.launch_count(reset=True)
    d_runs = 1.0 if prof["minors_d"][1] > 0 else 0.0
    st = Tb * cfg.volume
    if (flags & wk.CONTRACT_JACOBI) and prof["reduce"][1] == 0:
        # fused Jacobi kernel: propagators in, sigma out -- HBM bound by construction (4608 B per site-time)
        ms_k = prof["minors_u"][0]
        gbs = st * (4608.0 + 16.0) / (ms_k * 1e-3) / 1e9
        minors = {"bound": "hbm", "kernel": "jacobi_fused_kernel (a3-a5: two 12x12 inversions per site + complementary minors + term sum)",
                  "achieved": gbs, "peak": hbm_gbs, "unit": "GB/s", "frac": gbs / hbm_gbs if hbm_gbs else None,
                  "achieved_is": "4608 B of propagators + 16 B of sigma per site-time / CUDA-event time of the kernel",
                  "peak_source": "MEASURED_PEAKS.json hbm_gbs", "traffic": None, "launches_per_step": int(prof["minors_u"][1]),
                  "avg_launch_ms": ms_k / max(prof["minors_u"][1], 1), "kernel_share_of_step": ms_k / ms_step,
                  "note": "Jacobi complementary minors change the work, not only the rate: compare timeslices/s with the LU record, not FP64 %"}
        reduce, extra = None, {"project_ms_per_step": prof["project"][0]}
    else:
        minors, reduce, extra = rooflines(wk, cfg, terms, info, prof, ms_step, Tb, fp64_probe, hbm_gbs, d_runs)
    rec = {
        "workload": cfg.name, "contract_flags": int(flags), "isospin_u_equals_d": bool(isospin),
        "value": Tb / (ms_step * 1e-3), "unit": "timeslices/s", "ms_per_step": ms_step, "steps": steps,
        "timeslices_per_step": Tb, "L": cfg.L, "n_u": info.n_u, "n_d": info.n_d, "n_terms": int(info.n_terms),
        "unique_minors_per_site": int(info.n_minors_u + info.n_minors_d),
        "minor_dets_per_s": st * (info.n_minors_u + info.n_minors_d) / (ms_step * 1e-3),
        "minor_dets_per_s_kernel_only": st * (info.n_minors_u + d_runs * info.n_minors_d) / ((prof["minors_u"][0] + prof["minors_d"][0]) * 1e-3),
        "roofline": minors, "roofline_reduce": reduce, "gpu_launches": int(launches),
        "propagator_read_gbs": st * 4608 / (ms_step * 1e-3) / 1e9, **extra,
    }
    if clocks is not None:
        rec["clocks"] = clocks
    return rec, terms, (U, D, Cout)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=sorted(CONFIGS))
    ap.add_argument("--timeslices-per-step", type=int, default=4, help="contiguous timeslices per step and GPU (SURVEY 8(d): >= 4)")
    ap.add_argument("--ref-sites", type=int, default=1, help="oracle sites per step for --impl reference")
    ap.add_argument("--cpu-baseline-sites", type=int, default=1)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cpu-all-cores", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--side-workloads", default="cfg4,cfg4b", help="comma list measured in the same run and reported under "
                    "'workloads' (north_star names Li-7 next to He-4); '' to skip")
    ap.add_argument("--side-steps", type=int, default=400)
    ap.add_argument("--no-isospin-record", action="store_true", help="skip the extra U == D record of the headline workload")
    ap.add_argument("--isospin", action="store_true",
                    help="side measurement, not the headline: one propagator for both flavours (the paper's m_u = m_d, "
                         "PAPER.md:518); flavours with equal unique-minor tables then share one evaluation")
    args = ap.parse_args()
    cfg = CONFIGS[args.workload]
    if args.impl == "reference":
        run_reference(args, cfg)
        return

    import torch
    import torch.distributed as dist
    import paper_2411_08962_b200 as wk
    from paper_2411_08962_b200 import sharding
    from wick_inputs import make_propagators_torch

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the CUDA path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x: float) -> float:
        if world == 1:
            return x
        tt = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        return float(tt.item())

    hbm_gbs = read_measured_peaks().get("hbm_gbs")
    Tb = min(args.timeslices_per_step, max(cfg.T // world, 1))
    T_job = Tb * world                                        # weak scaling: Tb timeslices per GPU
    terms = workload_terms(wk, cfg)
    info = terms.info
    n_mom = len(cfg.momenta)
    # rank r owns the timeslices t = r (mod world) of the job's T_job timeslices (sharding.timeslices_of_rank);
    # no collective on the data path, one gather of C[p][t] at the end of every step
    mine = sharding.timeslices_of_rank(T_job, rank, world)
    parts = [make_propagators_torch(cfg.seed, cfg.L, cfg.T, dev, t0=t, nt=1) for t in mine]
    U = torch.cat([p[0] for p in parts]).contiguous()
    D = U if args.isospin else torch.cat([p[1] for p in parts]).contiguous()
    del parts
    ws = torch.empty(wk.contract_workspace_bytes(terms, cfg.L, len(mine), n_mom), dtype=torch.uint8, device=dev)
    result = {}

    def step():
        result["C"] = sharding.contract_sharded(U, D, terms, cfg.momenta, cfg.L, T_job, workspace=ws)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    fp64_probe = wk.measure_fp64_peak()

    # ---- timed region: K steps, profiling events off, device time via CUDA events on the launching stream ----
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    wk.launch_count(reset=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms_step = max_over_ranks(e0.elapsed_time(e1)) / args.steps
    launches = wk.launch_count(reset=True)
    clocks = sampler.stop() if rank == 0 else None
    value = T_job / (ms_step * 1e-3)
    C_dev = result["C"]

    # multi-GPU self-check: rank 0 recomputes a timeslice another rank owns and compares the gathered row bitwise
    shard_check = None
    if world > 1 and rank == 0:
        t_other = 1
        Uo, Do = make_propagators_torch(cfg.seed, cfg.L, cfg.T, dev, t0=t_other, nt=1)
        Co = wk.contract(Uo, Uo if args.isospin else Do, terms, cfg.momenta, cfg.L, 1)
        shard_check = bool(torch.equal(Co[:, 0], C_dev[:, t_other]))
        if not shard_check:
            raise RuntimeError("gathered C[p][t] differs from the single-rank result")

    # ---- separate pass: per-class kernel times (events around every launch) ----
    def local_step():
        wk.contract(U, D, terms, cfg.momenta, cfg.L, len(mine), workspace=ws)
    prof = class_times(wk, torch, local_step, max(1, min(3, args.steps)))
    wk.launch_count(reset=True)

    # ---- e2e: the same step through the host-buffer C-ABI call (H2D + D2H inside the timed region) ----
    e2e = None
    if not args.no_e2e:
        Uh = torch.empty(U.shape, dtype=U.dtype, pin_memory=True)
        Uh.copy_(U)
        if args.isospin:
            Dh = Uh
        else:
            Dh = torch.empty(D.shape, dtype=D.dtype, pin_memory=True)
            Dh.copy_(D)
        wk.contract_host(Uh, Dh, terms, cfg.momenta, cfg.L, len(mine))          # warm-up
        barrier()
        t_a = time.perf_counter()
        for _ in range(args.steps):
            C_host = wk.contract_host(Uh, Dh, terms, cfg.momenta, cfg.L, len(mine))   # synchronises before returning
        barrier()
        e2e_ms = max_over_ranks((time.perf_counter() - t_a) * 1e3 / args.steps)
        if not np.array_equal(C_host, C_dev[:, mine].cpu().numpy()):
            raise RuntimeError("host-buffer call disagrees with the device-buffer call")
        e2e = {"value": T_job / (e2e_ms * 1e-3), "unit": "timeslices/s",
               "h2d_bytes_per_step": int((1 if args.isospin else 2) * Uh.numel() * 16), "d2h_bytes_per_step": int(C_host.size * 16),
               "ms_per_step": e2e_ms, "timeslices_per_call": len(mine),
               "note": "wick_contract_host: timeslice blocks of <= 256 MB per flavour, H2D of block b+1 overlapped with the kernels of block b"}
        del Uh, Dh

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    d_runs = 1.0 if prof["minors_d"][1] > 0 else 0.0
    ms_step_local = ms_step
    minors, reduce, extra = rooflines(wk, cfg, terms, info, prof, ms_step_local, len(mine), fp64_probe, hbm_gbs, d_runs)
    st_per_step = len(mine) * cfg.volume
    minors_per_st = info.n_minors_u + info.n_minors_d

    # ---- side workloads (north_star: He-4 AND Li-7), rank 0's GPU, same run ----
    del U, D, ws
    torch.cuda.empty_cache()
    workloads = {}
    if world == 1:
        for key in [k for k in args.side_workloads.split(",") if k]:
            side_sampler = ClockSampler(local_rank)
            rec, _, _ = bench_workload(wk, torch, CONFIGS[key], key, args.timeslices_per_step, args.side_steps, args.warmup, dev,
                                       fp64_probe, hbm_gbs, sampler=side_sampler)
            if not args.no_cpu_baseline:
                rec["cpu_baseline"] = cpu_baseline_rows(CONFIGS[key], key, 4, False)
            workloads[CONFIGS[key].name] = rec
            torch.cuda.empty_cache()
            if CONFIGS[key].n_u >= 8 and CONFIGS[key].n_d >= 8:
                # the same workload through Jacobi's complementary-minor identity (opt-in flag)
                rec, _, _ = bench_workload(wk, torch, CONFIGS[key], key, args.timeslices_per_step, args.side_steps, args.warmup, dev,
                                           fp64_probe, hbm_gbs, flags=wk.CONTRACT_JACOBI)
                workloads[CONFIGS[key].name + "+jacobi"] = rec
                torch.cuda.empty_cache()
        if not cfg.random_list and cfg.n_u == cfg.n_d and not args.isospin and not args.no_isospin_record:
            # isospin limit of the headline workload (the paper's m_u = m_d): one propagator, one minor table,
            # swap-symmetrised factorised list
            rec, _, _ = bench_workload(wk, torch, cfg, args.workload, args.timeslices_per_step, max(args.steps, 2), args.warmup, dev,
                                       fp64_probe, hbm_gbs, isospin=True)
            rec["speedup_over_two_flavour_run"] = rec["value"] / value
            workloads[cfg.name + "+isospin"] = rec
            torch.cuda.empty_cache()
        if args.side_workloads:
            workloads["gevp_2x2_deuteron"] = bench_gevp(wk, torch, dev, args.timeslices_per_step, min(args.side_steps, 50), args.warmup)
            torch.cuda.empty_cache()

    cpu_baseline = None
    if not args.no_cpu_baseline:
        cpu_baseline = cpu_baseline_rows(cfg, args.workload, args.cpu_baseline_sites, not args.no_cpu_all_cores)

    line = {
        "metric": "correlator_timeslices_per_s", "value": value, "unit": "timeslices/s",
        "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64 (complex128)", "data": "synthetic",
        "config": {"workload": cfg.name, "L": cfg.L, "T": cfg.T, "timeslices_per_step": T_job, "timeslices_per_gpu": len(mine),
                   "n_u": info.n_u, "n_d": info.n_d,
                   "isospin_u_equals_d": bool(args.isospin), "n_terms": int(info.n_terms), "unique_minors_per_site": int(minors_per_st), "n_momenta": n_mom,
                   "l2_policy": "inputs_larger_than_l2 (and every site batch streams ~1.7 GB of minors through the 126 MB L2)",
                   "parallelism": f"timeslice shards t = r mod {world} (sharding.contract_sharded), no collective on the data path, one gather of C per step",
                   "profiling_events_in_timed_loop": False},
        "ms_per_timeslice": ms_step / len(mine),
        "minor_dets_per_s": world * st_per_step * minors_per_st / (ms_step * 1e-3),
        "minor_dets_per_s_kernel_only": st_per_step * (info.n_minors_u + d_runs * info.n_minors_d) / ((prof["minors_u"][0] + prof["minors_d"][0]) * 1e-3),
        "roofline": minors, "roofline_reduce": reduce, **extra,
        "cpu_baseline": cpu_baseline, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "hbm_peak_gbs_measured": hbm_gbs, "fp64_peak_tflops_measured": fp64_probe,
        "propagator_read_gbs": world * st_per_step * 4608 / (ms_step * 1e-3) / 1e9,
        "workloads": workloads, "sharded_result_bitwise_equal": shard_check,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
