#!/usr/bin/env python
"""bench.py — drag-update throughput (cells/s, fp64) of the fused CUDA path, with its roofline and the CPU oracle.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--no-sweep] [--legs] [--impl ours|reference]

A "step" is one pass of the whole hot path (a1..a5) over one batch of synthetic input = ONE
dg_drag_update launch over all cells of the workload.  Inputs are resident in HBM when the timed region starts;
out of place (p_out != p_in) so every launch does identical work; the working set (GBs) is far larger than the 126 MB
L2, so no L2 flush is needed between iterations.  Timing: CUDA events on the launching stream, barrier +
synchronize on both sides, max over ranks.  --gpus N > 1 runs N independent replicas (the path does not
shard, there is no collective on the data path); value = cells all ranks processed / max time.

Prints ONE short, strict-JSON line (rank 0; the last line of stdout, under 4 KB).  Keys beyond the base contract:
roofline, cpu_baseline, e2e, clocks, gpu_launches, peaks (the microbenchmarked denominators), ms_per_launch
(min / median / max over the timed launches), repeat_ms_per_step (two more timed regions of the same length: the
run-to-run spread) and a compact sweep (the other BASELINE.json configs, device-timed the same way: workload,
ms_per_step, bound, frac, timed_launches).  Everything else — the full per-workload records and, with --legs, the RK1 /
energy / single-precision / paper-as-printed measurements on the same buffers — goes to --detail-file
(default gpurun_out/bench_detail.json), never to stdout.
The default workload is BASELINE.json configs[3] (N = 16, 256^3 cells): the largest single-GPU configuration.
--impl reference times the CPU oracle (oracle/) on the host cores on the same workload recipe.
"""
import argparse
import json
import math
import os
import sys
import threading
import time

import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2509_25347_b200 import workloads as W  # noqa: E402

METRIC = "drag-update cells/sec (fp64)"
UNIT = "cells/s"
# Table B.1 for the ALGORITHMIC flop count of SURVEY.md §8(d): rows (m, Pi_m, theta_m)
TABLE_B1 = [(2, 1, 2.5809568e-8), (4, 2, 3.3971688e-4), (6, 3, 9.0656564e-3), (9, 4, 8.9577602e-2),
            (12, 5, 2.9961589e-1), (16, 6, 7.8028743e-1), (20, 7, 1.4382526), (25, 8, 2.4285825), (30, 9, 3.5396663)]
FP64_LANES_PER_SM = 64  # 4 sub-partitions x 16 fp64 FMA lanes (DESIGN.md §6 derives the ALU peak from this)


def algorithmic_bytes_per_cell(N):
    """read (2N+1) + 3(N+1) doubles, write 3(N+1) doubles = 8(8N+7) bytes."""
    return 8 * (8 * N + 7)


def algorithmic_flops(wl):
    """F = [min_k (Pi_mk + s_k)] * 2 n^3 + 6 n^2 per cell, s_k = max(0, ceil(log2(||A||_1/theta_mk))),
    summed over the workload's cells (the paper's own cost measure, B.11, times the dense product cost, plus the
    apply).  Returns (total flops, mean products per cell)."""
    n = wl.N + 1
    eps = wl.rho_d / wl.rho_g[None, :]
    a = wl.dt / wl.t_s
    norm = 2.0 * torch.maximum((eps * a).sum(dim=0), a.max(dim=0).values)
    best = None
    for m, pi, theta in TABLE_B1:
        s = torch.clamp(torch.ceil(torch.log2(norm / theta)), min=0.0)
        cost = s + pi
        best = cost if best is None else torch.minimum(best, cost)
    products = float(best.sum().item())
    return products * 2.0 * n ** 3 + 6.0 * n * n * wl.ncells, products / wl.ncells


def useful_flops(N, s, m):
    """Flops of the symmetric / sparse formulation of DESIGN.md §3 for the per-cell (m, s) the kernel reports, counted
    from the recurrences themselves (FMA = 2, add / mul / div / rsqrt = 1) and independent of the thread mapping: no
    padding, no divergence, no index or data-movement work.  This is the STRICT numerator of the ALU roofline: it can
    never exceed what the fp64 pipe executed, so the fraction can never exceed 1."""
    n = N + 1
    tri = n * (n - 1) // 2                       # strict upper triangle
    build = (1 + 2 * N) + 3 * N + (3 * N + 2)    # 1/rho_g, dt/t_s, eps; rsqrt, w; norm (N fma + max) and scaling
    first = 5 * N + (N * N + N)                  # al, be, be^2 (mul), b00 (N fma); P = (beta beta^T o U, beta o v) / m!
    horner = (1                                  # kappa_j = m!/j!
              + N * (N - 1)                      # U_ik <- v_k - alpha_i U_ik: one fma per packed dust entry
              + (2 * N - 1)                      # sum_l beta_l^2 v_l: one mul + (N-1) fma
              + 1 + 2 * N + 2)                   # kappa_j + Q_00; v_k <- x00 - alpha_k v_k (fma each); Q_00 (fma)
    conserve = (2 * N - 1) * n                   # per column: (N-1) fma and one mul
    square = n + tri * (1 + 2 * N) + conserve    # 1 + d; offdiag(X X): mul + N fma per entry; diagonal from conservation
    apply_ = 3 * (N + 2 * n * n + 1 + 2 * N)
    sm = s.double()
    mm = m.double()
    # thread-per-cell kernels with 6 <= N <= 10 leave the last squaring out and apply X_{s-1} twice (dg_tpc.cuh kDefer)
    kdef = 1 if 6 <= N <= 10 else 0
    deferred = sm.clamp(max=kdef)
    per_cell = (build + first + (mm - 1).clamp(min=0) * horner + tri + conserve + (sm - deferred) * square
                + torch.pow(2.0, deferred) * apply_)
    return float(per_cell.sum().item())


class ClockSampler:
    """SM clock, power and throttle reasons sampled through NVML every few ms WHILE the timed region runs
    (start() right before the first timed launch, stop() right after the closing synchronize)."""
    REASONS = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
               "hw_power_brake": 0x80}

    def __init__(self, device_index, period_s=0.004):
        self.period = period_s
        self.rows = []
        self.reasons = set()
        self.handle = None
        self.max_mhz = None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            try:
                uuid = str(torch.cuda.get_device_properties(device_index).uuid)
                self.handle = pynvml.nvmlDeviceGetHandleByUUID(uuid if uuid.startswith("GPU-") else "GPU-" + uuid)
            except Exception:
                self.handle = pynvml.nvmlDeviceGetHandleByIndex(device_index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.handle = None

    def _loop(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                mhz = nv.nvmlDeviceGetClockInfo(self.handle, nv.NVML_CLOCK_SM)
                mw = nv.nvmlDeviceGetPowerUsage(self.handle)
                mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.handle)
                self.rows.append((float(mhz), mw / 1000.0))
                for name, bit in self.REASONS.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        if self.handle is None:
            return
        self._stop.clear()
        self._thread = threading.Thread(target=self._loop, daemon=True)
        self._thread.start()

    def stop(self):
        if self._thread is not None:
            self._stop.set()
            self._thread.join(timeout=2)
            self._thread = None

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        sm = sorted(r[0] for r in self.rows)
        return {"sm_mhz": sm[len(sm) // 2], "sm_mhz_min": sm[0], "sm_max_mhz": self.max_mhz,
                "power_w_max": max(r[1] for r in self.rows), "reasons": sorted(self.reasons), "samples": len(sm)}


def aggregate_over_ranks(ms_local, cells_local):
    """max over ranks of the timed region, sum over ranks of the cells processed (the only cross-rank step)."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms_local), int(cells_local)
    dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else torch.device("cpu")
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=dev)
    c = torch.tensor([int(cells_local)], dtype=torch.int64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), int(c.item())


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


VARIANT = 0   # --variant: forces a thread mapping (dg_drag_update_variant) for mapping-against-mapping measurements


def _update(dg, wl, p_out):
    if VARIANT == 0:
        dg.dg_drag_update(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in, p_out=p_out)
    else:
        dg.dg_drag_update_ex(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in, p_out=p_out, variant=VARIANT)


def time_device_steps(dg, wl, p_out, steps, warmup, sampler=None, per_launch_events=True):
    """Returns (total ms over `steps` launches, list of per-launch ms).  The total is always one pair of CUDA events around
    the `steps` launches.  With per_launch_events an event is also recorded after every launch (per-launch minimum); an
    event between two launches costs the stream a few microseconds, which matters for the ~0.1 ms kernels of the sweep:
    those are timed without, and `per` is then the average repeated."""
    for _ in range(warmup):
        _update(dg, wl, p_out)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    barrier()
    torch.cuda.synchronize()
    if sampler is not None:
        sampler.start()
    ev[0].record()
    for k in range(steps):
        _update(dg, wl, p_out)
        if per_launch_events or k == steps - 1:
            ev[k + 1].record()
    torch.cuda.synchronize()
    if sampler is not None:
        sampler.stop()
    barrier()
    total = ev[0].elapsed_time(ev[steps])
    if per_launch_events:
        per = [ev[k].elapsed_time(ev[k + 1]) for k in range(steps)]
    else:
        per = [total / steps] * steps
    return total, per


def measure_peaks(dg, device, sm_count, sm_max_mhz):
    """The denominators MEASURED_PEAKS.json lacks: sustained DFMA / DMMA rates and an fp64 copy, one launch each timed
    with CUDA events (best of 5 after a warm-up)."""
    scratch = torch.empty(1 << 28, dtype=torch.float64, device=device)  # 2 GiB: copy 1 GiB -> 1 GiB
    scratch.zero_()
    out = {}
    for name, kind, iters in (("dfma_tflops", 0, 20000), ("dmma_tflops", 1, 20000), ("dfma_dmma_mixed_tflops", 2, 5000),
                              ("fp64_copy_gbs", 3, 1)):
        best = None
        for rep in range(6):
            e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
            e0.record()
            work = dg.dg_peak_kernel(kind, iters, scratch)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            if rep > 0:
                best = ms if best is None else min(best, ms)
        out[name] = work / (best * 1e-3) / (1e9 if kind == 3 else 1e12)
    del scratch
    out["fp64_nominal_tflops"] = sm_count * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
    return out


def measured_peaks_file():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback (B200_PROFILING.md)"


def ncu_traffic(workload):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch, from the committed ncu --set full summary of this
    workload (profiles/traffic.csv: workload,kernel,dram_read_bytes,dram_write_bytes,source), or None."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        for ln in f:
            c = ln.strip().split(",")
            if len(c) >= 4 and c[0] == workload:
                return float(c[2]) + float(c[3])
    return None


def roofline_for(wl, ms_per_launch, dense_flops, flops, peaks, hbm_gbs, hbm_src):
    """The binding roofline of the fused kernel: whichever of (algorithmic bytes / HBM peak) and (algorithmic flops /
    fp64 ALU peak) takes longer.  `flops` is the strict count of useful_flops(); `dense_flops` is SURVEY.md §8(d)'s
    dense-product figure F (what Alg. 6-7 of the paper would execute), reported beside it as `dense_equivalent`."""
    nbytes = algorithmic_bytes_per_cell(wl.N) * wl.ncells
    peak = peaks["fp64_nominal_tflops"]
    t_hbm = nbytes / (hbm_gbs * 1e9)
    t_alu = flops / (peak * 1e12)
    sec = ms_per_launch * 1e-3
    dense = {"achieved": dense_flops / sec / 1e12, "unit": "TFLOP/s", "frac": dense_flops / sec / 1e12 / peak,
             "note": "SURVEY.md 8(d) F = [min_k(Pi_mk + s_k)] 2n^3 + 6n^2: the flops of the paper's dense Alg. 6-7; "
                     "the kernels execute fewer (symmetric squarings, sparse Horner), so this can exceed 1"}
    traffic = ncu_traffic(wl.name)
    if t_alu >= t_hbm:
        ach = flops / sec / 1e12
        return {"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                "traffic": traffic, "algorithmic_bytes": nbytes,
                "flops": "useful flops of the symmetric/sparse formulation for the per-cell (m, s) (DESIGN.md §6)",
                "peak_source": "nominal fp64 FMA peak = SMs x 64 lanes x 2 x clocks.max.sm (DESIGN.md §6); "
                               "measured DFMA microbenchmark in peaks.dfma_tflops",
                "frac_of_measured_dfma": ach / peaks["dfma_tflops"],
                "hbm_frac": (nbytes / sec / 1e9) / hbm_gbs, "dense_equivalent": dense}
    ach = nbytes / sec / 1e9
    return {"bound": "hbm", "achieved": ach, "peak": hbm_gbs, "unit": "GB/s", "frac": ach / hbm_gbs,
            "traffic": traffic, "algorithmic_bytes": nbytes, "peak_source": hbm_src,
            "alu_frac": (flops / sec / 1e12) / peak, "dense_equivalent": dense}


def cpu_oracle_sample(wl, budget_s=15.0):
    """Times the oracle as it stands (all host threads) on a strided sample of the workload sized for ~budget_s."""
    from oracle import dgo
    threads = dgo.max_threads()

    def run(nsample, nthreads=0):
        idx = W.sample_cells(wl.ncells, nsample)
        rho_g, rho_d, t_s, p_in = wl.cells(idx)
        t0 = time.perf_counter()
        dgo.drag_update(rho_g, rho_d, t_s, wl.dt, p_in, nthreads=nthreads)
        return len(idx), time.perf_counter() - t0

    dgo.lib()
    nc, sec = run(min(wl.ncells, 2048))                     # calibration
    rate = nc / max(sec, 1e-6)
    nsample = int(min(wl.ncells, max(2048, rate * budget_s)))
    nc, sec = run(nsample)
    n1, sec1 = run(int(min(wl.ncells, max(1024, rate / threads * 3.0))), nthreads=1)   # ~3 s on one core
    return {"value": nc / sec, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"{nc} cells strided over the {wl.ncells}-cell workload, {sec:.1f} s",
            "value_1core": n1 / sec1, "sample_1core": f"{n1} cells, {sec1:.1f} s"}


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, same workload recipe, each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import dgo
    wl = W.make_workload(args.config, ncells=min(W.CONFIG_CELLS[args.config], 1 << 20), N=args.N, device="cpu")
    threads = dgo.max_threads()
    dgo.lib()
    idx = W.sample_cells(wl.ncells, 2048)
    cells = wl.cells(idx)
    t0 = time.perf_counter(); dgo.drag_update(cells[0], cells[1], cells[2], wl.dt, cells[3]); cal = time.perf_counter() - t0
    total_budget = 120.0
    per_step = total_budget / (args.steps + args.warmup)
    nsample = int(min(wl.ncells, max(1024, len(idx) / max(cal, 1e-6) * per_step)))
    idx = W.sample_cells(wl.ncells, nsample)
    cells = wl.cells(idx)
    for _ in range(args.warmup):
        dgo.drag_update(cells[0], cells[1], cells[2], wl.dt, cells[3])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        dgo.drag_update(cells[0], cells[1], cells[2], wl.dt, cells[3])
    sec = time.perf_counter() - t0
    value = len(idx) * args.steps / sec
    full_cells = W.CONFIG_CELLS[args.config]
    sample = (f"{len(idx)} cells per step, strided over a {wl.ncells}-cell draw of the same recipe "
              f"(the workload itself has {full_cells} cells)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f80 (x87 long double)", "data": "synthetic",
        "config": {"workload": f"config{args.config}_N{wl.N}_{full_cells}cells",
                   "recipe": f"BASELINE.json configs[{args.config - 1}]", "N": wl.N, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}, allow_nan=False))


def bench_rk1(dg, wl, p_out, hbm_gbs, steps=5, warmup=3):
    """The first-order implicit RK1 step (dg_drag_rk1, App. A.2) on the same buffers: the
    paper's speed reference for EXP (Fig. 6-7).  Same algorithmic bytes per cell, O(N) flops: HBM roofline."""
    for _ in range(warmup):
        dg.dg_drag_rk1(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in, p_out=p_out)
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(steps):
        dg.dg_drag_rk1(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in, p_out=p_out)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    gbs = algorithmic_bytes_per_cell(wl.N) * wl.ncells / (ms * 1e-3) / 1e9
    return {"ms_per_launch": ms, "cells_per_s": wl.ncells / (ms * 1e-3), "bound": "hbm", "achieved_gbs": gbs,
            "hbm_frac": gbs / hbm_gbs}


def _timed_ms(f, steps, warmup):
    for _ in range(warmup):
        f()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(steps):
        f()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / steps


def bench_energy(dg, wl, p_out, ms_update, hbm_gbs, steps=5, warmup=2):
    """dg_drag_update_energy (Eq. 4, R20): ONE launch of the default kernel for N, which
    forms the kinetic-energy sums from the values its apply step holds anyway — algorithmic bytes per cell 8(8N+7) + 16
    (E read and written)."""
    E_in = torch.ones(wl.ncells, dtype=torch.float64, device=wl.rho_g.device)
    E_out = torch.empty_like(E_in)
    ms = _timed_ms(lambda: dg.dg_drag_update_energy(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in, E_in, 0.5, p_out=p_out,
                                                    E_out=E_out), steps, warmup)
    total = algorithmic_bytes_per_cell(wl.N) + 16
    return {"ms_per_launch_sequence": ms, "launches": 1, "cells_per_s": wl.ncells / (ms * 1e-3),
            "over_plain_update": ms / ms_update, "algorithmic_bytes_per_cell": total,
            "hbm_frac": total * wl.ncells / (ms * 1e-3) / 1e9 / hbm_gbs}


def bench_f32(dg, wl, ms_update, fp32_peak_tflops, steps=5, warmup=2):
    """dg_drag_update_f32 (Eq. B.8 with u = 2^-24) on the same fields rounded to float: useful flops
    of ITS (m, s) against the fp32 FMA peak (128 lanes per SM), and the time against the fp64 path."""
    f = lambda t: t.to(torch.float32).contiguous()
    rho_g, rho_d, t_s, p_in = f(wl.rho_g), f(wl.rho_d), f(wl.t_s), f(wl.p_in)
    out = torch.empty_like(p_in)
    _, s, m = dg.dg_drag_update_f32(rho_g, rho_d, t_s, wl.dt, p_in, p_out=out)
    ms = _timed_ms(lambda: dg.dg_drag_update_f32(rho_g, rho_d, t_s, wl.dt, p_in, p_out=out), steps, warmup)
    flops = useful_flops(wl.N, s, m)
    peak = fp32_peak_tflops
    tf = flops / (ms * 1e-3) / 1e12
    hbm = 4 * (8 * wl.N + 7) * wl.ncells / (ms * 1e-3) / 1e9
    return {"ms_per_launch": ms, "cells_per_s": wl.ncells / (ms * 1e-3), "achieved_tflops": tf, "fp32_peak_tflops": peak,
            "alu_frac": tf / peak, "achieved_gbs": hbm, "mean_s": float(s.double().mean().item()),
            "mean_m": float(m.double().mean().item()), "fp64_over_f32_time": ms_update / ms}


def bench_paper_variant(dg, wl, p_out, steps=2, warmup=1):
    """The paper's own scheme as printed (one thread per cell, dense matrices, Alg. 7 + plain squarings; SURVEY.md
    §8(f) rank 3) on the same buffers, for the design comparison on the same hardware: with the row chosen by
    min(Pi_m + s) (DG_VARIANT_PAPER), by Algorithm 2 as printed (DG_VARIANT_PAPER_ALG2), and with Algorithm 2 plus the
    bound test of Algorithms 8-9 (DG_VARIANT_PAPER_BOUND: products saved per cell = (m - m_evaluated) / q)."""
    def timed(variant):
        f = lambda: dg.dg_drag_update_ex(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in, p_out=p_out, variant=variant)
        for _ in range(warmup):
            f()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(steps):
            _, s, m = f()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / steps, s, m
    ms, s0, m0 = timed(dg.DG_VARIANT_PAPER)
    drift = ((p_out.sum(dim=1) - wl.p_in.sum(dim=1)).abs() / wl.p_in.abs().sum(dim=1)).max().item()
    res = {"ms_per_launch": ms, "cells_per_s": wl.ncells / (ms * 1e-3), "max_momentum_drift": drift}
    pi = {2: 1, 4: 2, 6: 3, 9: 4, 12: 5, 16: 6, 20: 7, 25: 8, 30: 9}
    qq = {2: 1, 4: 2, 6: 2, 9: 3, 12: 3, 16: 4, 20: 4, 25: 5, 30: 5}
    pi_t = torch.zeros(31, dtype=torch.float64, device=s0.device); q_t = torch.ones(31, dtype=torch.float64, device=s0.device)
    for k, v in pi.items():
        pi_t[k] = v; q_t[k] = qq[k]
    cost = lambda s, m: float((pi_t[m.long()] + s.double()).mean().item())
    res["mean_products_min_cost"] = cost(s0, m0)
    if wl.ncells > (1 << 22):   # the two further variants cost seconds per launch at N = 16: 2^22-cell workloads only
        return res
    steps, warmup = 1, (1 if ms < 100.0 else 0)   # seconds per launch at N >= 12: no warm-up needed there
    ms2, s2, m2 = timed(dg.DG_VARIANT_PAPER_ALG2)
    # Alg. 7 recomputes the powers inside every block: r(q-1) + (r-1) dense products, not Pi_m = q + r - 2
    rr = {2: 2, 4: 2, 6: 3, 9: 3, 12: 4, 16: 4, 20: 5, 25: 5, 30: 6}
    a7_t = torch.zeros(31, dtype=torch.float64, device=s0.device)
    for k in pi:
        a7_t[k] = rr[k] * (qq[k] - 1) + (rr[k] - 1)
    cost7 = lambda s, m: float((a7_t[m.long()] + s.double()).mean().item())
    res["mean_products_alg7_min_cost"] = cost7(s0, m0)
    res["alg2"] = {"ms_per_launch": ms2, "mean_products": cost(s2, m2), "mean_products_alg7": cost7(s2, m2)}
    ms3, s3, m3 = timed(dg.DG_VARIANT_PAPER_BOUND)
    saved = ((m2 - m3).double() / q_t[m2.long()]).mean().item()
    res["alg2_bound_test"] = {"ms_per_launch": ms3, "mean_products_saved_by_bound_test": float(saved)}
    return res


def bench_one(dg, wl, steps, warmup, peaks, hbm_gbs, hbm_src, sampler=None, min_region_ms=0.0, legs=False, repeats=0):
    """One workload, device-timed.  min_region_ms > 0 (the sweep entries): the number of timed launches is raised (up to
    400) until the timed region lasts about that long, and no event is recorded between launches — a 0.1 ms kernel timed
    over five launches with an event after each reads 5-8 % slow (launch latency after the synchronize, event gaps)."""
    p_out = torch.empty_like(wl.p_in)
    fine = True
    if min_region_ms > 0.0:
        t_est, _ = time_device_steps(dg, wl, p_out, 3, warmup, None, per_launch_events=False)
        want = int(math.ceil(min_region_ms / max(t_est / 3, 1e-3)))
        if want > steps:
            steps, fine = min(want, 400), False
    total_ms, per = time_device_steps(dg, wl, p_out, steps, warmup, sampler, per_launch_events=fine)
    dense_flops, products = algorithmic_flops(wl)
    _, s, m = dg.dg_drag_update_ex(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in, p_out=p_out, variant=VARIANT)  # untimed: per-cell (m, s)
    flops = useful_flops(wl.N, s, m)
    ms_launch = sum(per) / len(per)
    roof = roofline_for(wl, ms_launch, dense_flops, flops, peaks, hbm_gbs, hbm_src)
    sp = sorted(per)
    res = {"workload": wl.name, "N": wl.N, "ncells": wl.ncells, "ms_per_step": total_ms / steps,
           # per-launch figures exist only where an event was recorded after every launch (not in the sweep entries)
           "ms_per_launch": {"min": sp[0], "median": sp[len(sp) // 2], "max": sp[-1]} if fine else None,
           "timed_launches": steps, "cells_per_s": wl.ncells * steps / (total_ms * 1e-3),
           "useful_flops_per_cell": flops / wl.ncells, "dense_flops_per_cell": dense_flops / wl.ncells,
           "dense_products_per_cell": products, "algorithmic_bytes_per_cell": algorithmic_bytes_per_cell(wl.N),
           "mean_s": float(s.double().mean().item()), "mean_m": float(m.double().mean().item()),
           "max_s": int(s.max().item()), "roofline": roof, "variant": dg.dg_variant_name(wl.N)}
    # the run-to-run spread: further timed regions of the same length, after the one the headline is taken from
    res["repeat_ms_per_step"] = [time_device_steps(dg, wl, p_out, steps, 1, None, per_launch_events=fine)[0] / steps
                                 for _ in range(repeats)]
    if legs:   # --legs: the SURVEY.md §8(f) entry points on the same buffers (detail file only)
        res["rk1"] = bench_rk1(dg, wl, p_out, hbm_gbs, steps=5 if fine else max(5, steps))   # same timed-region rule
        res["rk1"]["exp_over_rk1_time"] = ms_launch / res["rk1"]["ms_per_launch"]
        if wl.ncells <= (1 << 22):   # the two rank-4 entry points, on the 2^21..2^22-cell workloads (they need extra buffers)
            res["energy"] = bench_energy(dg, wl, p_out, ms_launch, hbm_gbs)
            res["f32"] = bench_f32(dg, wl, ms_launch, 2.0 * peaks["fp64_nominal_tflops"])   # 128 fp32 vs 64 fp64 FMA lanes per SM
        res["paper_as_printed"] = bench_paper_variant(dg, wl, p_out)
        res["paper_as_printed"]["speedup_of_product_path"] = res["paper_as_printed"]["ms_per_launch"] / ms_launch
    del p_out
    return res, total_ms


def _strict(x):
    """A copy of x that json.dumps(..., allow_nan=False) accepts: non-finite floats become None."""
    if isinstance(x, float):
        return x if math.isfinite(x) else None
    if isinstance(x, dict):
        return {k: _strict(v) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_strict(v) for v in x]
    return x


def _rounded(x, digits=6):
    """Floats to `digits` significant digits (the printed line only: the detail file keeps full precision)."""
    if isinstance(x, float):
        return float(f"{x:.{digits}g}") if math.isfinite(x) else x
    if isinstance(x, dict):
        return {k: _rounded(v, digits) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_rounded(v, digits) for v in x]
    return x


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json configs[config-1] (default 4: N = 16, 256^3, the "
                    "largest single-GPU configuration); 5 = sweep point (give --N)")
    ap.add_argument("--N", type=int, default=None)
    ap.add_argument("--variant", type=int, default=0, help="force a mapping: 1 thread/cell, 2 warp/cell DMMA, 4 pair/cell")
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--legs", action="store_true", help="also time RK1 / energy / f32 / paper-as-printed (detail file only)")
    ap.add_argument("--detail-file", default=os.path.join(ROOT, "gpurun_out", "bench_detail.json"))
    args = ap.parse_args()
    if args.config == 5 and args.N is None:
        args.N = 16
    if args.impl == "reference":
        run_reference(args)
        return
    global VARIANT
    VARIANT = args.variant

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)
    from paper_2509_25347_b200 import binding as dg  # raises if libdg.so is missing

    props = torch.cuda.get_device_properties(device)
    mp_file, hbm_src = measured_peaks_file()
    hbm_gbs = float(mp_file["hbm_gbs"])
    sm_max_mhz = float(mp_file.get("sm_max_mhz", 1965.0))
    peaks = measure_peaks(dg, device, props.multi_processor_count, sm_max_mhz)

    # replicas: every rank runs the same recipe with its own seed
    wl = W.make_workload(args.config, N=args.N, device=device, seed=rank)
    clk = ClockSampler(local_rank)
    res, total_ms = bench_one(dg, wl, args.steps, args.warmup, peaks, hbm_gbs, hbm_src, sampler=clk, legs=args.legs,
                              repeats=2)
    clocks = clk.summary()
    ms_max, cells_all = aggregate_over_ranks(total_ms, wl.ncells * args.steps)
    value = cells_all / (ms_max * 1e-3)

    # end to end through the host-buffer C-ABI call: pinned host tensors -> H2D -> kernel -> D2H, every step
    e2e = None
    if not args.no_e2e:
        n = wl.N + 1
        host = [t.cpu().pin_memory() for t in (wl.rho_g, wl.rho_d, wl.t_s, wl.p_in)]
        h_out = torch.empty_like(host[3]).pin_memory()
        e2e_steps = max(1, min(args.steps, 3))
        dg.dg_drag_update_host(host[0], host[1], host[2], wl.dt, host[3], p_out=h_out)  # warm-up (allocates staging)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            dg.dg_drag_update_host(host[0], host[1], host[2], wl.dt, host[3], p_out=h_out)
        sec = time.perf_counter() - t0
        barrier()
        ms_e2e, cells_e2e = aggregate_over_ranks(sec * 1e3, wl.ncells * e2e_steps)
        e2e = {"value": cells_e2e / (ms_e2e * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": 8 * (1 + 2 * wl.N + 3 * n) * wl.ncells, "d2h_bytes_per_step": 8 * 3 * n * wl.ncells,
               "steps": e2e_steps, "api": "dg_drag_update_host (pinned host buffers, chunked, 3 streams)"}
        dg.dg_host_release()
        del host, h_out

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_oracle_sample(wl)

    sweep = []
    if rank == 0 and world == 1 and not args.no_sweep:
        del wl
        torch.cuda.empty_cache()
        points = [(c, None) for c in (2, 3, 4) if c != args.config] + [(5, N) for N in W.SWEEP_N]
        for cfg, N in points:
            w2 = W.make_workload(cfg, N=N, device=device)
            r2, _ = bench_one(dg, w2, max(3, min(args.steps, 5)), 3, peaks, hbm_gbs, hbm_src, min_region_ms=20.0,
                              legs=args.legs)
            sweep.append(r2)
            del w2
            torch.cuda.empty_cache()

    if rank == 0:
        roof = res["roofline"]
        short_roof = {k: roof.get(k) for k in ("bound", "achieved", "peak", "unit", "frac", "traffic", "algorithmic_bytes")}
        short_roof["peak_source"] = ("nominal fp64 FMA peak = SMs x 64 lanes x 2 x clocks.max.sm (DESIGN.md §6)"
                                     if roof["bound"] == "alu" else hbm_src)
        if roof["bound"] == "alu":
            short_roof["flops_per_cell"] = res["useful_flops_per_cell"]
            short_roof["frac_of_measured_dfma"] = roof["frac_of_measured_dfma"]
            short_roof["dense_equivalent_frac"] = roof["dense_equivalent"]["frac"]
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": res["workload"], "recipe": f"BASELINE.json configs[{args.config - 1}]",
                       "N": res["N"], "ncells_per_gpu": res["ncells"], "parallelism": "replicas" if world > 1 else "1 GPU",
                       "l2": "inputs larger than L2 (no flush)", "variant": res["variant"]},
            "roofline": short_roof, "cpu_baseline": cpu, "e2e": e2e, "clocks": clocks,
            "gpu_launches": args.steps * dg.dg_launches_per_update(res["N"], res["ncells"]),
            "ms_per_launch": res["ms_per_launch"], "repeat_ms_per_step": res["repeat_ms_per_step"],
            "peaks": dict(peaks, hbm_gbs=hbm_gbs, hbm_source=hbm_src, gpu=props.name, sms=props.multi_processor_count),
            "sweep": [{"workload": r["workload"], "ms_per_step": r["ms_per_step"], "bound": r["roofline"]["bound"],
                       "frac": r["roofline"]["frac"], "timed_launches": r["timed_launches"]} for r in sweep],
        }
        line = _strict(_rounded(line))
        detail = _strict({"line": line, "headline": res, "sweep": sweep,
                          "paper_context": "A100/Dyablo N=8: 9.7e-9 s/cell = 1.03e8 cells/s (PAPER.md:341); other machine"})
        try:
            os.makedirs(os.path.dirname(args.detail_file), exist_ok=True)
            with open(args.detail_file, "w") as f:
                json.dump(detail, f, indent=1, allow_nan=False)
        except OSError as e:   # a read-only checkout must not cost the headline
            print(f"bench.py: could not write {args.detail_file}: {e}", file=sys.stderr)
        text = json.dumps(line, allow_nan=False, separators=(",", ":"))
        if len(text) > 4000:   # the driver keeps only the tail of stdout: the sweep is in the detail file anyway
            line["sweep"] = []
            text = json.dumps(line, allow_nan=False, separators=(",", ":"))
        sys.stdout.flush()
        print(text, flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
