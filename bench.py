#!/usr/bin/env python
"""bench.py -- throughput of the determinant-form Wick contraction hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg3]

A "step" is one pass of the whole hot path (steps a3-a6 of DESIGN.md: propagator staging, unique minor
determinants, weighted products, momentum projection) over one batch of synthetic input: the FULL term
list of the workload on `timeslices_per_step` full timeslices of its lattice.  Default workload: cfg3
(Helium-4, L = 32, 2716 x 2716 terms, 858,050 unique 6x6 minors per site), the configuration
BASELINE.json's target is quoted on.  Metric: correlator timeslices/s (whole job); the same run also
reports unique minor dets/s and the FP64 roofline fraction of the dominant kernel.

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

def executed_flops_per_site(n: int, row_in_order: np.ndarray, cols_in_order: np.ndarray) -> float:
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


def oracle_seconds_per_site(cfg, n_sites: int):
    """Time the oracle (MERGED mode = the paper's method A, two fresh determinants per term) on
    n_sites sites of the workload.  Returns (seconds per site, threads used)."""
    from oracle import wick_oracle as wo
    U, D = make_propagators_numpy(cfg.seed, cfg.L, cfg.T, t0=0, nt=1)
    if cfg.random_list:
        lst = make_random_term_list(cfg.seed, cfg.n_u, cfg.n_d, cfg.n_random_terms)
        run = lambda s: wo.site_terms_value(U[0, s], D[0, s], *lst)
    else:
        sink = wo.merged_terms(cfg.nucleus)
        run = lambda s: wo.site_value_outer(U[0, s], D[0, s], sink)
    t0 = time.perf_counter()
    for s in range(n_sites):
        run(s)
    return (time.perf_counter() - t0) / n_sites, 1          # numpy elementwise code: one thread


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


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=sorted(CONFIGS))
    ap.add_argument("--timeslices-per-step", type=int, default=1)
    ap.add_argument("--ref-sites", type=int, default=1, help="oracle sites per step for --impl reference")
    ap.add_argument("--cpu-baseline-sites", type=int, default=2)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
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

    Tb = min(args.timeslices_per_step, cfg.T)
    terms = workload_terms(wk, cfg)
    info = terms.info
    n_mom = len(cfg.momenta)
    # weak scaling: every rank owns its own block of Tb timeslices (shard by timeslice, no exchange)
    t0_slice = (rank * Tb) % max(cfg.T - Tb + 1, 1)
    U, D = make_propagators_torch(cfg.seed, cfg.L, cfg.T, dev, t0=t0_slice, nt=Tb)
    if args.isospin:
        D = U
    ws = torch.empty(wk.contract_workspace_bytes(terms, cfg.L, Tb, n_mom), dtype=torch.uint8, device=dev)
    Cout = torch.empty((n_mom, Tb), dtype=torch.complex128, device=dev)

    def step():
        wk.contract(U, D, terms, cfg.momenta, cfg.L, Tb, workspace=ws, out=Cout)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    fp64_probe = wk.measure_fp64_peak()

    # ---- timed region: K steps, device time via CUDA events on the launching stream ----
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    wk.launch_count(reset=True)
    wk.profile_enable(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = wk.launch_count(reset=True)
    prof = wk.profile_read()
    wk.profile_enable(False)
    clocks = sampler.stop() if rank == 0 else None
    if world > 1:
        tt = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        ms_total = float(tt.item())
    ms_step = ms_total / args.steps
    value = world * Tb / (ms_step * 1e-3)

    # ---- e2e: the same step through the host-buffer C-ABI call (H2D + D2H inside the timed region) ----
    e2e = None
    if not args.no_e2e:
        Uh = torch.empty(U.shape, dtype=U.dtype, pin_memory=True)
        Dh = torch.empty(D.shape, dtype=D.dtype, pin_memory=True)
        Uh.copy_(U)
        Dh.copy_(D)
        wk.contract_host(Uh, Dh, terms, cfg.momenta, cfg.L, Tb)          # warm-up
        barrier()
        t_a = time.perf_counter()
        for _ in range(args.steps):
            C_host = wk.contract_host(Uh, Dh, terms, cfg.momenta, cfg.L, Tb)   # synchronises before returning
        barrier()
        e2e_ms = (time.perf_counter() - t_a) * 1e3 / args.steps
        if world > 1:
            tt = torch.tensor([e2e_ms], dtype=torch.float64, device=dev)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            e2e_ms = float(tt.item())
        if not np.allclose(C_host, Cout.cpu().numpy(), rtol=1e-12, atol=0):
            raise RuntimeError("host-buffer call disagrees with the device-buffer call")
        e2e = {"value": world * Tb / (e2e_ms * 1e-3), "unit": "timeslices/s",
               "h2d_bytes_per_step": int(2 * Uh.numel() * 16), "d2h_bytes_per_step": int(C_host.size * 16),
               "ms_per_step": e2e_ms}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (a4: minors_kernel<n_u>, minors_kernel<n_d>) ----
    st_per_step = Tb * cfg.volume
    minors_per_st = info.n_minors_u + info.n_minors_d
    d_runs = 1.0 if prof["minors_d"][1] > 0 else 0.0           # isospin: the d minors may be served by the u table
    flop_minors = st_per_step * (info.n_minors_u * flops_lu(info.n_u) + d_runs * info.n_minors_d * flops_lu(info.n_d))
    ms_minors = (prof["minors_u"][0] + prof["minors_d"][0]) / args.steps
    ms_reduce = prof["reduce"][0] / args.steps
    ms_project = prof["project"][0] / args.steps
    n_minor_launches = (prof["minors_u"][1] + prof["minors_d"][1]) // args.steps
    achieved_tf = flop_minors / (ms_minors * 1e-3) / 1e12
    mu_row, _, md_row, _ = terms.minors()
    ou, od = terms.minor_order(0), terms.minor_order(1)
    exec_site = (executed_flops_per_site(info.n_u, mu_row[ou[0]], ou[1]), executed_flops_per_site(info.n_d, md_row[od[0]], od[1]))
    executed_tf = st_per_step * (exec_site[0] + d_runs * exec_site[1]) / (ms_minors * 1e-3) / 1e12
    traffic = None
    try:
        with open(os.path.join(ROOT, "profiles", "r01_roofline_traffic.json.txt")) as f:
            traffic = json.load(f).get(cfg.name, {}).get("minors_dram_bytes_per_launch")
    except Exception:
        pass
    roofline = {
        "bound": "alu", "kernel": " / ".join({6: "minors6_cached_kernel", 10: "minors_large_cached_kernel<10>", 11: "minors_large_cached_kernel<11>"}.get(n, f"minors_kernel<{n}>") for n in (info.n_u, info.n_d))
                                  + " (a4, LU with partial pivoting)",
        "achieved": achieved_tf, "peak": FP64_PEAK_DERIVED_TFLOPS, "unit": "TFLOP/s",
        "frac": achieved_tf / FP64_PEAK_DERIVED_TFLOPS,
        "peak_source": "derived: 148 SMs x 64 FP64 lanes x 2 flop x 1.965 GHz (MEASURED_PEAKS.json has no FP64 entry)",
        "executed": {"tflops": executed_tf, "frac": executed_tf / FP64_PEAK_DERIVED_TFLOPS,
                     "flops_per_minor": {"u": exec_site[0] / max(info.n_minors_u, 1), "d": exec_site[1] / max(info.n_minors_d, 1)},
                     "note": "flops the kernel issues: LU state shared by minors with equal row tuple and leading columns "
                             "(DESIGN.md 6b); `achieved`/`frac` count one full LU per unique minor (SURVEY 8d) and can exceed 1"},
        "peak_measured_dfma_probe": fp64_probe, "frac_of_dfma_probe": achieved_tf / fp64_probe if fp64_probe else None,
        "traffic": traffic, "launches_per_step": int(n_minor_launches),
        "avg_launch_ms": ms_minors / max(n_minor_launches, 1),
        "algorithmic_flops_per_minor": {"u": flops_lu(info.n_u), "d": flops_lu(info.n_d)},
        "kernel_share_of_step": ms_minors / ms_step,
        "reduce": {"ms_per_step": ms_reduce, "tflops": st_per_step * info.n_terms * FLOPS_PER_TERM / (ms_reduce * 1e-3) / 1e12
                   if ms_reduce > 0 else None, "share_of_step": ms_reduce / ms_step},
        "project_ms_per_step": ms_project,
        "per_flavour": {
            q: {"n": n, "ms_per_step": prof[k][0] / args.steps,
                "frac": (st_per_step * nm * flops_lu(n) / (prof[k][0] / args.steps * 1e-3) / 1e12 / FP64_PEAK_DERIVED_TFLOPS)
                if prof[k][0] > 0 else None}
            for q, k, n, nm in (("u", "minors_u", info.n_u, info.n_minors_u), ("d", "minors_d", info.n_d, info.n_minors_d))},
        "whole_step_tflops": (flop_minors + st_per_step * info.n_terms * FLOPS_PER_TERM) / (ms_step * 1e-3) / 1e12,
    }

    cpu_baseline = None
    if not args.no_cpu_baseline:
        sps, cores = oracle_seconds_per_site(cfg, args.cpu_baseline_sites)
        cpu_baseline = {"value": 1.0 / (sps * cfg.volume), "unit": "timeslices/s", "cores": cores, "kind": "oracle",
                        "sample": f"{args.cpu_baseline_sites} sites of {cfg.name} (full term list), {sps:.2f} s per site, "
                                  f"scaled by L^3 = {cfg.volume} sites per timeslice",
                        "host_cores_available": len(os.sched_getaffinity(0))}

    line = {
        "metric": "correlator_timeslices_per_s", "value": value, "unit": "timeslices/s",
        "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64 (complex128)", "data": "synthetic",
        "config": {"workload": cfg.name, "L": cfg.L, "T": cfg.T, "timeslices_per_step": Tb, "n_u": info.n_u, "n_d": info.n_d,
                   "isospin_u_equals_d": bool(args.isospin), "n_terms": int(info.n_terms), "unique_minors_per_site": int(minors_per_st), "n_momenta": n_mom,
                   "l2_policy": "inputs_larger_than_l2" if 2 * U.numel() * 16 > 126e6 else "working_set_larger_than_l2",
                   "parallelism": f"timeslice shards x{world}, no collective on the data path"},
        "minor_dets_per_s": world * st_per_step * minors_per_st / (ms_step * 1e-3),
        "minor_dets_per_s_kernel_only": st_per_step * (info.n_minors_u + d_runs * info.n_minors_d) / (ms_minors * 1e-3),
        "roofline": roofline, "cpu_baseline": cpu_baseline, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "hbm_peak_gbs_measured": read_measured_peaks().get("hbm_gbs"),
        "propagator_read_gbs": st_per_step * 4608 / (ms_step * 1e-3) / 1e9,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
