#!/usr/bin/env python
"""bench.py -- one "step" = one pass of the whole hot path (pattern
count, scan, column indices, FP64 fill, then the workload's P0*x products) over one synthetic
lattice.  Default workload: BASELINE.json configs[4] ("cfg5", the largest single-GPU configuration: nd channels
J = 1/2 .. 7/2, both parities, pair j <= 3, N_p = N_q = 150 tan^2 grid, 10-point Gauss-Legendre, 20 SpMVs per
J^pi matrix; 1.67e10 nonzeros per step, one matrix of up to 39 GB resident at a time).  Prints ONE JSON line
(contract in the task statement).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg1..cfg5] [--impl reference] [--only-jpi 7,-1]

N > 1 (torchrun): the path shards over independent problems, no data-path collective.  The nd workloads deal their
J^pi matrices to the ranks (largest first, to the least loaded rank; total work fixed: "scaling": "strong"); the
s-wave workloads give every rank its own lattice (seed + rank; "scaling": "weak").
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import wpcd_inputs as wi  # noqa: E402

# DRAM bytes per launch of the dominant kernel from one `ncu --set full` capture (dram__bytes_read.sum +
# dram__bytes_write.sum), profiles/r01h_ncu_full.md; null where no capture of that workload exists.
NCU_TRAFFIC = {
    ("cfg2", "spmv"): 3.84e6,            # spmv_kernel<32,4>, one pass of 4 right-hand sides over the 3.4 MB matrix (cold L2 under ncu; r01h)
    ("cfg2", "fill_swave"): 6.88e6,
    ("cfg4", "spmv"): 6.19e9,            # r01h: CSR product, J^pi = 1/2+ matrix (5.14e8 nnz): 6.17 GB algorithmic
    # profiles/r02_ncu_full.md: one launch on the J^pi = 7/2- matrix (3.24e9 nonzeros, the largest of the eight)
    ("cfg5", "spmv"): 26.29e9,           # spmv_georow_kernel<1,256>: 26.27 GB read + 0.02 GB written; algorithmic 26.40 GB for that matrix
    ("cfg5", "fill_coupled"): 0.787e9,   # contract_kernel, one chunk of 16 000 elements: 0.680 GB written + 0.107 GB read; 0.703 GB algorithmic
}
NCU_TRAFFIC_NOTE = {
    ("cfg5", "spmv"): "launch on the J^pi = 7/2- matrix (3.24e9 nnz; 26.40 GB algorithmic for that launch, the step's mean launch is smaller)",
    ("cfg5", "fill_coupled"): "contract_kernel, one 16 000-element chunk of the J^pi = 7/2- matrix (0.703 GB algorithmic); the moments stay in L2",
}

METRIC = "P-matrix nonzeros/sec (FP64 build + the workload's P*vector SpMVs per step)"
UNIT = "nnz/s"
FLOPS_PER_NODE = 70.0          # algorithmic FP64 flops per (phi,x) quadrature node, s-wave
L2_FLUSH_BYTES = 256 << 20     # > 126 MB L2


# --------------------------------------------------------------------------- helpers
def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0}, "fallback"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.reasons, self.sm_max = index, False, [], set(), None
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {
            nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
            nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
        }
        while not self.stop_flag:
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.01)

    def summary(self):
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.sm_max,
                "reasons": sorted(self.reasons), "samples": len(self.sm)}


def jobs_of(wl):
    """[(two_J, parity)] per step; the s-wave workloads have one (dummy) job."""
    return wl.jpis if wl.model == "nd" else [(0, 0)]


# --------------------------------------------------------------------------- reference arm (oracle on host cores)
def oracle_tables(wl):
    from oracle import channels as och
    from oracle import perm as operm

    tabs = []
    for (two_J, parity) in jobs_of(wl):
        if wl.model == "swave":
            ch, pairs = och.spinless_swave_table(wl.g0)
        else:
            ch = och.enumerate_channels(two_J, parity, wl.j_pair_max)
            pairs = och.g_table(ch, two_J, 1)
        tabs.append(operm.PairTable(ch, pairs))
    return tabs


def oracle_pass(wl, tabs, row_stride):
    """One bounded oracle pass: full pattern, values on every row_stride-th geometric row (all
    channels), the workload's SpMVs on the s-wave workloads.  Returns (nnz_evaluated, seconds)."""
    from oracle import perm as operm

    p = wl.grid()
    t0 = time.perf_counter()
    geo = operm.geo_pattern(p, p)
    n_geo = wl.n_bins * wl.n_bins
    rows = np.arange(0, n_geo, row_stride)
    done = 0
    for tab in tabs:
        if wl.model == "swave":
            rp, ci, v, _ = operm.build_csr(p, p, wl.n_quad, tab, geo=geo)
            done += len(v)
            for k in range(wl.n_spmv):
                operm.spmv(rp, ci, v, wi.normal_vector(len(rp) - 1, k=k))
        else:
            cnt = (geo[0][rows + 1] - geo[0][rows])
            erow = np.repeat(rows, cnt)
            eidx = np.concatenate([np.arange(geo[0][r], geo[0][r + 1]) for r in rows])
            ecol = geo[1][eidx]
            n_q = wl.n_bins
            val, _ = operm.element_values(p, p, erow // n_q, erow % n_q, ecol // n_q, ecol % n_q, wl.n_quad, tab)
            done += val.size
    return done, time.perf_counter() - t0


def reference_row_stride(wl):
    # bounded oracle sample, sized for roughly 5-30 s of CPU work on a 16-core host
    return {"cfg1": 1, "cfg2": 1, "cfg3": 1, "cfg4": 24, "cfg5": 64, "fig4": 1}[wl.name]


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import perm as operm

    wl = wi.WORKLOADS[args.workload]
    tabs = oracle_tables(wl)
    stride = reference_row_stride(wl)
    for _ in range(max(args.warmup, 0) and 1):
        oracle_pass(wl, tabs, stride)
    steps = max(1, min(args.steps, 5))
    t, nnz = 0.0, 0
    for _ in range(steps):
        n, dt = oracle_pass(wl, tabs, stride)
        t += dt
        nnz += n
    value = nnz / t
    sample = (f"full {wl.name} pass (pattern + values + {wl.n_spmv} SpMV)" if stride == 1
              else f"full pattern + values of every {stride}th geometric row, all channel pairs")
    cores = operm.num_threads()
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": 1 if args.warmup else 0, "ms_per_step": 1e3 * t / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "n_bins": wl.n_bins, "n_quad": wl.n_quad, "model": wl.model, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# --------------------------------------------------------------------------- our arm
class Job:
    """One (J, parity) matrix.  Device buffers are views into a pool shared by all jobs of the
    step (sized for the largest), so only one matrix is resident at a time (DESIGN.md memory plan)."""

    def __init__(self, channels, rows):
        self.channels, self.rows = channels, rows
        self.nnz = self.nnz_geo = 0
        self.graph = None


def allocate(wpcd, torch, grid, jobs, wl):
    n_geo = grid.n_p * grid.n_q
    max_rows = max(j.rows for j in jobs)
    row_ptr = torch.empty(max_rows + 1, dtype=torch.int64, device="cuda")
    geo_row_ptr = torch.empty(n_geo + 1, dtype=torch.int32, device="cuda")
    ws_bytes = 256
    for j in jobs:
        j.row_ptr, j.geo_row_ptr = row_ptr[: j.rows + 1], geo_row_ptr
        j.nnz, j.nnz_geo = wpcd.wpcd_perm_count(grid, j.channels, wl.n_quad, j.row_ptr, j.geo_row_ptr)
        ws_bytes = max(ws_bytes, wpcd.wpcd_perm_workspace_bytes(j.channels, j.nnz_geo))
    max_nnz = max(j.nnz for j in jobs)
    col_idx = torch.empty(max_nnz, dtype=torch.int32, device="cuda")
    values = torch.empty(max_nnz, dtype=torch.float64, device="cuda")
    workspace = torch.empty(ws_bytes, dtype=torch.uint8, device="cuda")
    n_x = max(1, wl.n_spmv) if wl.model == "swave" else max(1, min(wl.n_spmv, 4))
    x_host = torch.from_numpy(np.stack([wi.normal_vector(max_rows, k=k) for k in range(n_x)])).pin_memory()
    x = x_host.cuda()
    y = torch.empty(max_rows, dtype=torch.float64, device="cuda")
    y_host = torch.empty(max_rows, dtype=torch.float64).pin_memory()
    for j in jobs:
        j.col_idx, j.values, j.workspace = col_idx[: j.nnz], values[: j.nnz], workspace
        j.n_x = n_x
        j.x = [x[k, : j.rows] for k in range(n_x)]
        j.x_host = [x_host[k, : j.rows] for k in range(n_x)]
        j.y, j.y_host = y[: j.rows], y_host[: j.rows]
        # s-wave workloads keep all n_spmv vectors (one job, rows == max_rows): the end-to-end leg hands them to
        # the library in ONE host call
        j.x_all, j.x_host_all = (x, x_host) if (wl.model == "swave" and n_x == wl.n_spmv and j.rows == max_rows) else (None, None)
    if jobs[0].x_all is not None:
        jobs[0].y_all = torch.empty_like(x)
        jobs[0].y_host_all = torch.empty(x_host.shape, dtype=torch.float64).pin_memory()


def run_ours(args):
    import torch

    from paper_1404_5253_b200 import build as _build

    from paper_1404_5253_b200 import shard

    rank, local_rank, world = shard.rank_world()
    if rank == 0:
        _build.build()
    import paper_1404_5253_b200 as wpcd

    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist.barrier()
    wpcd.load()
    wl = wi.WORKLOADS[args.workload]
    strong = wl.model == "nd"          # nd sweeps: the J^pi matrices of ONE lattice are dealt to the ranks
    p = wl.grid(seed_offset=0 if strong else shard.lattice_seed_offset(rank))   # s-wave: independent lattice per rank (weak scaling)
    grid = wpcd.wpcd_grid_create(p, p)

    def make_channels(two_J, parity):
        if wl.model == "swave":
            return wpcd.wpcd_channels_create(wpcd.WPCD_SPINLESS_SWAVE, g0=wl.g0)
        return wpcd.wpcd_channels_create(wpcd.WPCD_ND, two_J=two_J, parity=parity, two_T=1, j_pair_max=wl.j_pair_max)

    # one J^pi matrix resident at a time; buffers sized for the largest
    all_jpis = jobs_of(wl)
    if args.only_jpi:
        tj, par = (int(v) for v in args.only_jpi.split(","))
        all_jpis = [jp for jp in all_jpis if tuple(jp) == (tj, par)]
        assert all_jpis, "--only-jpi names no matrix of this workload"
    all_ch = [make_channels(two_J, parity) for (two_J, parity) in all_jpis]
    # cost of a matrix ~ its coupled channel pairs (the geometric pattern is shared): largest first, to the least loaded rank
    mine = shard.assign_balanced(list(range(len(all_jpis))), [c.pairs for c in all_ch], rank, world) if strong else list(range(len(all_jpis)))
    my_jpis = [all_jpis[k] for k in mine]
    jobs = [Job(all_ch[k], wpcd.wpcd_rows(grid, all_ch[k])) for k in mine]
    idle = not jobs                    # more ranks than matrices: this rank only takes part in the reductions
    if not idle:
        allocate(wpcd, torch, grid, jobs, wl)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device="cuda")
    # count / build of a job with their arguments marshalled once (fixed buffers, fixed stream): the Python side of a step is
    # two ctypes calls per job
    for job in jobs:
        job.count, job.build = wpcd.bind_count_build(grid, job.channels, wl.n_quad, job.row_ptr, job.geo_row_ptr, job.workspace,
                                                     job.col_idx, job.values, torch.cuda.current_stream())
    n_spmv = wl.n_spmv

    def spmv_sweep(job):
        if job.x_all is not None:
            # all right-hand sides of the workload are resident (s-wave workloads; P is reused for many energies):
            # one call, the library shares each pass over the matrix among 4 of them
            wpcd.wpcd_perm_apply(job.rows, job.row_ptr, job.col_idx, job.values, job.x_all, job.y_all, n_vec=n_spmv)
            return
        # coupled channels: the product through the block structure of P0 (same CSR arrays, values streamed only: 8 B per nonzero)
        for k in range(n_spmv):
            wpcd.wpcd_perm_apply_blocked(grid, job.channels, job.row_ptr, job.geo_row_ptr, job.col_idx, job.values, job.x[k % job.n_x], job.y)

    def sweep_passes(job):
        """[right-hand sides per launch] of one sweep (mirrors the library: passes of 4, then 2, then 1)."""
        if job.x_all is None:
            return [1] * n_spmv
        out, v = [], 0
        while v < n_spmv:
            step_v = 4 if n_spmv - v >= 4 else 2 if n_spmv - v >= 2 else 1
            out.append(step_v)
            v += step_v
        return out

    def step(job_list):
        for job in job_list:
            job.count()
            job.build()
            if n_spmv:
                if job.graph is not None:
                    job.graph.replay()
                else:
                    spmv_sweep(job)

    # capture the launch-bound SpMV sweep in a CUDA graph (small matrices only)
    if not idle:
        step(jobs)
    torch.cuda.synchronize()
    if n_spmv and wl.model == "swave":
        for job in jobs:
            g = torch.cuda.CUDAGraph()
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                spmv_sweep(job)
            torch.cuda.current_stream().wait_stream(side)
            torch.cuda.synchronize()
            with torch.cuda.graph(g):
                spmv_sweep(job)
            job.graph = g
    for _ in range(args.warmup if not idle else 0):
        step(jobs)
    torch.cuda.synchronize()
    fp64_peak = wpcd.wpcd_fp64_peak()

    # ---- timed region: device-resident inputs
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank)
    sampler.start()
    launches0 = wpcd.wpcd_launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for s in range(args.steps):
        flush.fill_(s & 0xFF)                       # L2 flush between timed iterations (not timed)
        ev[s][0].record()
        for job in jobs:
            job.count()
            job.build()
            if n_spmv:
                if job.graph is not None:
                    job.graph.replay()
                else:
                    spmv_sweep(job)
        ev[s][1].record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    graph_launches = sum(len(sweep_passes(job)) for job in jobs if job.graph is not None) * args.steps
    launches = wpcd.wpcd_launch_count() - launches0 + graph_launches
    # ---- the same steps once more with CUDA events around every stage (the library's stage trace) and around the sweep: the
    # per-stage and per-launch times of the rooflines.  Kept out of the region above because the events themselves cost
    # ~17 us per step on the small workloads (5 % of the cfg2 step).
    inst_steps = max(1, min(args.steps, 20 if wl.model == "swave" else 3))
    wpcd.wpcd_trace_enable(True)
    wpcd.wpcd_trace_read()
    sp_ev = []
    for s in range(inst_steps):
        flush.fill_(s & 0xFF)
        for job in jobs:
            job.count()
            job.build()
            if n_spmv:
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                if job.graph is not None:
                    job.graph.replay()
                else:
                    spmv_sweep(job)
                b.record()
                sp_ev.append((a, b))
    torch.cuda.synchronize()
    stages = wpcd.wpcd_trace_read()
    wpcd.wpcd_trace_enable(False)
    sampler.stop_flag = True
    sampler.join()
    total_ms = sum(a.elapsed_time(b) for a, b in ev)
    spmv_ms = sum(a.elapsed_time(b) for a, b in sp_ev)
    ms_max, nnz_all = shard.reduce_step(dist, "cuda", total_ms, sum(j.nnz for j in jobs))
    ms_per_step = ms_max / args.steps
    value = shard.throughput(ms_per_step, nnz_all)
    extras = rank == 0 and not idle and not args.no_extras

    # ---- extra: multi-vector apply: 4 right-hand sides share one pass over the matrix
    spmm = None
    if n_spmv and extras:
        job = jobs[-1]                     # its matrix is the one resident after the timed region
        x4 = torch.from_numpy(np.stack([wi.normal_vector(job.rows, k=100 + k) for k in range(4)])).cuda().contiguous()
        y4 = torch.empty_like(x4)
        for _ in range(3):
            wpcd.wpcd_perm_apply(job.rows, job.row_ptr, job.col_idx, job.values, x4, y4, n_vec=4)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 20 if wl.model == "swave" else 5
        a.record()
        for _ in range(reps):
            wpcd.wpcd_perm_apply(job.rows, job.row_ptr, job.col_idx, job.values, x4, y4, n_vec=4)
        b.record()
        torch.cuda.synchronize()
        ms4 = a.elapsed_time(b) / reps
        spmm = {"n_vec": 4, "ms_per_pass": ms4, "products_per_s": 4.0 / (ms4 * 1e-3),
                "matrix_GBps": (12.0 * job.nnz + 8.0 * job.rows) / (ms4 * 1e-3) / 1e9, "nnz": job.nnz}
        # complex right-hand side (the transition operator is complex): one 16-byte gather, two FMAs per entry
        xc = torch.complex(x4[0], x4[1]).contiguous()
        yc = torch.empty_like(xc)
        for _ in range(3):
            wpcd.wpcd_perm_apply_complex(job.rows, job.row_ptr, job.col_idx, job.values, xc, yc)
        a.record()
        for _ in range(reps):
            wpcd.wpcd_perm_apply_complex(job.rows, job.row_ptr, job.col_idx, job.values, xc, yc)
        b.record()
        torch.cuda.synchronize()
        msc = a.elapsed_time(b) / reps
        spmm["complex_ms_per_product"] = msc
        spmm["complex_matrix_GBps"] = (12.0 * job.nnz + 8.0 * job.rows) / (msc * 1e-3) / 1e9
        # four real vectors interleaved [rows][4]: one 32-byte gather per entry
        xi4 = x4.t().contiguous()
        yi4 = torch.empty_like(xi4)
        for _ in range(3):
            wpcd.wpcd_perm_apply_interleaved(job.rows, job.row_ptr, job.col_idx, job.values, xi4, yi4)
        a.record()
        for _ in range(reps):
            wpcd.wpcd_perm_apply_interleaved(job.rows, job.row_ptr, job.col_idx, job.values, xi4, yi4)
        b.record()
        torch.cuda.synchronize()
        msi = a.elapsed_time(b) / reps
        spmm["interleaved4_ms_per_pass"] = msi
        spmm["interleaved4_matrix_GBps"] = (12.0 * job.nnz + 8.0 * job.rows) / (msi * 1e-3) / 1e9
        # the general CSR product (12 B per nonzero) and the product through the block structure of P0 (8 B per nonzero), one vector
        for name, fn in (("csr", lambda: wpcd.wpcd_perm_apply(job.rows, job.row_ptr, job.col_idx, job.values, x4[0], y4[0])),
                         ("blocked", lambda: wpcd.wpcd_perm_apply_blocked(grid, job.channels, job.row_ptr, job.geo_row_ptr, job.col_idx,
                                                                          job.values, x4, y4, n_vec=1))):
            for _ in range(2):
                fn()
            a.record()
            for _ in range(reps):
                fn()
            b.record()
            torch.cuda.synchronize()
            spmm[name + "_ms_per_product"] = a.elapsed_time(b) / reps
        spmm["csr_matrix_GBps"] = (12.0 * job.nnz + 24.0 * job.rows) / (spmm["csr_ms_per_product"] * 1e-3) / 1e9
        spmm["blocked_matrix_GBps"] = (8.0 * job.nnz + 16.0 * job.rows) / (spmm["blocked_ms_per_product"] * 1e-3) / 1e9
        # many right-hand sides (P0 is reused for ~100 energies): 8 vectors share one pass of the blocked product
        x8 = torch.from_numpy(np.stack([wi.normal_vector(job.rows, k=200 + k) for k in range(8)])).cuda().contiguous()
        y8 = torch.empty_like(x8)
        for nv in (2, 4, 8):
            for _ in range(2):
                wpcd.wpcd_perm_apply_blocked(grid, job.channels, job.row_ptr, job.geo_row_ptr, job.col_idx, job.values, x8, y8, n_vec=nv)
            a.record()
            for _ in range(reps):
                wpcd.wpcd_perm_apply_blocked(grid, job.channels, job.row_ptr, job.geo_row_ptr, job.col_idx, job.values, x8, y8, n_vec=nv)
            b.record()
            torch.cuda.synchronize()
            spmm["blocked_nvec%d_ms_per_pass" % nv] = a.elapsed_time(b) / reps
        del x8, y8
        # one application of the factored kernel K = O P0 O^T V1 G1 (synthetic O, V1, G1)
        n_ch = job.channels.count
        o_h, v_h, g_h = wi.kernel_factors(n_ch, grid.n_p, grid.n_q)
        o_d, v_d, g_d = torch.from_numpy(o_h).cuda(), torch.from_numpy(v_h).cuda(), torch.from_numpy(g_h).cuda()
        scratch = torch.empty(2 * job.rows, dtype=torch.complex128, device="cuda")
        for _ in range(2):
            wpcd.wpcd_kernel_apply(n_ch, grid.n_p, grid.n_q, job.row_ptr, job.col_idx, job.values, o_d, v_d, g_d, xc, yc, scratch)
        a.record()
        for _ in range(reps):
            wpcd.wpcd_kernel_apply(n_ch, grid.n_p, grid.n_q, job.row_ptr, job.col_idx, job.values, o_d, v_d, g_d, xc, yc, scratch)
        b.record()
        torch.cuda.synchronize()
        spmm["kernel_apply_ms"] = a.elapsed_time(b) / reps
        spmm["kernel_apply_dense_gflop"] = 3 * 2.0 * n_ch * grid.n_p ** 2 * (2 * grid.n_q) / 1e9

        # the dependent products of the iteration in one call (wpcd_perm_apply_chain): small matrices only
        if wl.model == "swave":
            n_it = 50
            ych = torch.empty(n_it, job.rows, dtype=torch.float64, device="cuda")
            for _ in range(3):
                wpcd.wpcd_perm_apply_chain(job.rows, job.row_ptr, job.col_idx, job.values, x4[0], ych, n_it)
            a.record()
            for _ in range(5):
                wpcd.wpcd_perm_apply_chain(job.rows, job.row_ptr, job.col_idx, job.values, x4[0], ych, n_it)
            b.record()
            torch.cuda.synchronize()
            spmm["chain50_us_per_product"] = a.elapsed_time(b) / 5 / n_it * 1e3

    # ---- extra: the kink-split rule RS(n) (R14): cost of the build against R(n)
    rule_split = {}
    job = jobs[-1] if not idle else None
    rules = [("plain", wl.n_quad), ("split", wl.n_quad | wpcd.WPCD_RULE_KINK_SPLIT)] if extras else []
    if wl.model == "swave":
        rules += [("analytic_u", wl.n_quad | wpcd.WPCD_RULE_ANALYTIC_U), ("analytic_u_n32", 32 | wpcd.WPCD_RULE_ANALYTIC_U), ("plain_n32", 32)]
    for name, nq in rules:
        reps = 3 if wl.model == "swave" else 1
        for _ in range(1):
            wpcd.wpcd_perm_build(grid, job.channels, nq, job.row_ptr, job.geo_row_ptr, job.workspace, job.col_idx, job.values)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            wpcd.wpcd_perm_build(grid, job.channels, nq, job.row_ptr, job.geo_row_ptr, job.workspace, job.col_idx, job.values)
        b.record()
        torch.cuda.synchronize()
        rule_split["build_ms_" + name] = a.elapsed_time(b) / reps
    if extras:
        wpcd.wpcd_perm_build(grid, job.channels, wl.n_quad, job.row_ptr, job.geo_row_ptr, job.workspace, job.col_idx, job.values)
    torch.cuda.synchronize()

    # ---- end to end through the C-ABI with HOST buffers (handles, tables and vectors from the host)
    # The channel handle of the next J^pi (host g-table of (A4), a few tens of ms) is made by a helper thread while the GPU
    # works on the current matrix: the library calls release the GIL, handle creation touches no state of other handles.
    from concurrent.futures import ThreadPoolExecutor
    helper = ThreadPoolExecutor(max_workers=1)

    def e2e_step():
        g2 = wpcd.wpcd_grid_create(p, p)
        threaded = wl.model == "nd" and len(my_jpis) > 1
        ahead = helper.submit(make_channels, *my_jpis[0]) if threaded else None
        for k_job, job in enumerate(jobs):
            ch2 = ahead.result() if threaded else make_channels(*my_jpis[k_job])
            if threaded and k_job + 1 < len(my_jpis):
                ahead = helper.submit(make_channels, *my_jpis[k_job + 1])
            wpcd.wpcd_perm_count(g2, ch2, wl.n_quad, job.row_ptr, job.geo_row_ptr)
            wpcd.wpcd_perm_build(g2, ch2, wl.n_quad, job.row_ptr, job.geo_row_ptr, job.workspace, job.col_idx, job.values)
            if n_spmv and job.x_all is not None:      # the independent vectors are known up front: one host call, n_vec = n_spmv
                wpcd.wpcd_perm_apply_host(job.rows, job.row_ptr, job.col_idx, job.values, job.x_host_all, job.y_host_all,
                                          job.x_all, job.y_all, n_vec=n_spmv)
                continue
            for k in range(n_spmv):
                wpcd.wpcd_perm_apply_blocked_host(g2, ch2, job.row_ptr, job.geo_row_ptr, job.col_idx, job.values, job.x_host[k % job.n_x],
                                                  job.y_host, job.x[0], job.y)
    e2e_steps = max(1, min(args.steps, 20 if wl.model == "swave" else 3))
    e2e_step()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    torch.cuda.synchronize()
    e2e_s = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(e2e_s, op=dist.ReduceOp.MAX)
    e2e_value = nnz_all / (e2e_s.item() / e2e_steps)
    table_bytes = sum(12 * j.channels.terms + 8 * j.channels.pairs + 16 * j.channels.count for j in jobs)
    h2d = 2 * 8 * (wl.n_bins + 1) + table_bytes + sum(8 * j.rows * n_spmv for j in jobs)
    d2h = sum(8 * j.rows * n_spmv + 4 for j in jobs)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- rooflines (per launch; stage and sweep times from the instrumented repeat).  Algorithmic work per unit is
    # SURVEY.md section 8(d)'s, restated in DESIGN.md section 7.
    peaks, peak_kind = measured_peaks()
    nnz1 = sum(j.nnz for j in jobs)
    nnz_geo1 = sum(j.nnz_geo for j in jobs)
    rows1 = sum(j.rows for j in jobs)
    steps = inst_steps          # the stage and sweep times below come from the instrumented repeat
    roofs = {}
    stage_ms = {k: v[0] / steps for k, v in stages.items()}
    hbm_src = f"MEASURED_PEAKS.json hbm_gbs ({peak_kind})"
    alu_src = "in-run DFMA microbenchmark (wpcd_fp64_peak)"
    if stage_ms["fill_swave"] > 0:
        flops = FLOPS_PER_NODE * wl.n_quad * wl.n_quad * nnz1
        ach = flops / (stage_ms["fill_swave"] * 1e-3) / 1e12
        roofs["fill_swave"] = {"bound": "alu", "achieved": ach, "peak": fp64_peak / 1e12, "unit": "TFLOP/s",
                               "frac": ach / (fp64_peak / 1e12), "traffic": None, "ms_per_launch": stage_ms["fill_swave"],
                               "peak_source": alu_src}
    t_fill = (stage_ms["moments"] + stage_ms["contract"]) * 1e-3
    if t_fill > 0:
        # two bounds, the larger one is the roofline: the HBM write of 12 B per nonzero (value + column index), and the
        # FP64 work of schedule (B) of SURVEY 8(d): per geometric element n^2 nodes x 2 flops x n_mu monomial moments,
        # plus 2 flops per (pair, monomial) coefficient of the g-contraction
        wbytes = 12.0 * nnz1
        flops = sum(j.nnz_geo * (2.0 * wl.n_quad * wl.n_quad * j.channels.monomials + 2.0 * j.channels.coefficients) for j in jobs)
        t_hbm, t_alu = wbytes / (peaks["hbm_gbs"] * 1e9), flops / fp64_peak
        hbm = {"bound": "hbm", "achieved": wbytes / t_fill / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
               "frac": t_hbm / t_fill, "peak_source": hbm_src}
        alu = {"bound": "alu", "achieved": flops / t_fill / 1e12, "peak": fp64_peak / 1e12, "unit": "TFLOP/s",
               "frac": t_alu / t_fill, "peak_source": alu_src}
        top = dict(hbm if t_hbm >= t_alu else alu)
        top.update({"traffic": None, "both_bounds": {"hbm": hbm, "alu": alu},
                    "ms_per_step": {"moments": stage_ms["moments"], "contract": stage_ms["contract"]},
                    "algorithmic": {"bytes": wbytes, "flops": flops}})
        roofs["fill_coupled"] = top
    if n_spmv:
        # algorithmic bytes of a launch with v right-hand sides: the matrix once + v vectors in and out.  The CSR product
        # (s-wave workloads) reads 12 B per nonzero + row_ptr; the blocked product (coupled channels) reads the values only,
        # 8 B per nonzero, the geometric pattern (4 B per geometric entry) and x once per (channel, geometric entry)
        blocked = wl.model == "nd"
        n_launch = sum(len(sweep_passes(j)) for j in jobs)
        if blocked:
            sbytes = sum(sum(8.0 * j.nnz + 4.0 * j.nnz_geo + v * (8.0 * j.channels.count * j.nnz_geo + 8.0 * j.rows) for v in sweep_passes(j))
                         for j in jobs)
        else:
            sbytes = sum(sum(12.0 * j.nnz + 8.0 * j.rows + v * 16.0 * j.rows for v in sweep_passes(j)) for j in jobs)
        csr_bytes = sum(sum(12.0 * j.nnz + 8.0 * j.rows + v * 16.0 * j.rows for v in sweep_passes(j)) for j in jobs)
        per_launch_ms = spmv_ms / (steps * n_launch)
        ach = sbytes / (spmv_ms / steps * 1e-3) / 1e9
        roofs["spmv"] = {"bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": ach / peaks["hbm_gbs"],
                         "traffic": None, "ms_per_launch": per_launch_ms, "launches_per_step": n_launch,
                         "rhs_per_launch": max(max(sweep_passes(j)) for j in jobs),
                         "kernel_name": "spmv_georow_kernel<1,256> (wpcd_perm_apply_blocked)" if blocked else "spmv_kernel (wpcd_perm_apply)",
                         "algorithmic_bytes_per_step": sbytes,
                         "csr_equivalent_GBps": csr_bytes / (spmv_ms / steps * 1e-3) / 1e9,
                         "peak_source": hbm_src,
                         "note": "matrix is L2-resident (3 MB)" if wl.model == "swave" else "values stream from HBM, 8 B per nonzero"}
    share = dict(stage_ms)
    share["spmv_sweep"] = spmv_ms / steps
    # the selection (a1-a3) is reported by its time only (latency-bound, no per-unit figure)
    kernels = {"fill_swave": "fill_swave", "moments": "fill_coupled", "contract": "fill_coupled", "spmv_sweep": "spmv"}
    dominant = max((k for k in share if k in kernels), key=share.get)
    key = kernels[dominant]
    for name, rf in roofs.items():
        rf["traffic"] = NCU_TRAFFIC.get((wl.name, name))
        if (wl.name, name) in NCU_TRAFFIC_NOTE:
            rf["traffic_launch"] = NCU_TRAFFIC_NOTE[(wl.name, name)]
    roofline = dict(roofs[key]) if key in roofs else {
        "bound": "alu", "achieved": None, "peak": fp64_peak / 1e12, "unit": "TFLOP/s", "frac": None, "traffic": None}
    roofline["kernel"] = dominant

    # ---- oracle on the host cores beside it (N = 1 only)
    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        from oracle import perm as operm

        stride = reference_row_stride(wl)
        n, dt = oracle_pass(wl, oracle_tables(wl), stride)
        cpu_baseline = {"value": n / dt, "unit": UNIT, "cores": operm.num_threads(), "kind": "oracle",
                        "sample": (f"full {wl.name} pass (pattern + values + {wl.n_spmv} SpMV), {dt:.1f} s" if stride == 1 else
                                   f"full pattern + values of every {stride}th geometric row, all channel pairs, {dt:.1f} s")}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong" if strong else "weak", "vs_baseline": None,
        "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": wl.name, "n_bins": wl.n_bins, "n_quad": wl.n_quad, "model": wl.model, "jitter": wl.jitter,
                   "jpis": all_jpis if wl.model == "nd" else None, "n_spmv_per_matrix": n_spmv,
                   "nnz": int(nnz_all), "nnz_rank0": nnz1, "nnz_geo_rank0": nnz_geo1, "rows_rank0": rows1,
                   "sharding": ("J^pi matrices dealt to the ranks, largest first" if strong else "one lattice per rank") if world > 1 else "none",
                   "l2": "flushed between timed steps (256 MiB fill)",
                   "spmv_launch": ("CUDA graph" if jobs[0].graph is not None else "direct")
                   + (", one call for all right-hand sides (passes of 4)" if jobs[0].x_all is not None and n_spmv else "")},
        "clocks": sampler.summary(),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "steps": e2e_steps, "includes": "grid/channel handle creation (host g-table; the next J^pi's on a helper thread), count, build, the products with pinned-host x and y"
                            + (" (one wpcd_perm_apply_host call with n_vec = %d: the vectors are independent and known up front)" % n_spmv
                               if (not idle and jobs[0].x_all is not None and n_spmv) else " (one wpcd_perm_apply_blocked_host call per product)")},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "rooflines": roofs,
        "stage_ms_per_step": share,
        "build_nnz_per_s": nnz1 / max(1e-12, (ms_per_step - spmv_ms / steps) * 1e-3),
        "stage_timing": f"instrumented repeat of {inst_steps} steps after the timed region (events around every stage)",
        "fp64_peak_tflops_measured": fp64_peak / 1e12,
        "spmm_nvec4": spmm, "rule_split": rule_split,
        "cpu_baseline": cpu_baseline,
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg5", choices=sorted(wi.WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the untimed extra measurements (multi-vector products, rule variants)")
    ap.add_argument("--only-jpi", default="", help="two_J,parity: restrict an nd workload to one matrix (profiling runs)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
