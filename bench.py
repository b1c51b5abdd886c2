#!/usr/bin/env python
"""bench.py — k-points/s of the whole hot path (bs_assemble + bs_bands over every k-point of one workload).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5] [--impl ours|reference]

A "step" is one pass of the whole path (S1..S8 of DESIGN.md) over one workload: assembly of Phi/Psi and their
factors, then the lowest `nbands` eigenvalues at every k-point.  `value` = k-points per second with the inputs already
resident on the device; `e2e` = the same through the public API with HOST buffers (bs_create_cell copies the geometry
in, bs_bands copies omega^2 out) inside the timed region.  Under torchrun each rank owns an interleaved share of a
k-path N times denser (weak scaling, no data-path collective: DESIGN.md section 8); the line also carries `strong`: the
SAME k-path split contiguously over the ranks by paper_1310_6380_b200.sharded, with the all-gather of the results.
The default run (N = 1, C5) then runs C1-C4 for a few steps each and reports them under `all_configs`.
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
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

import workloads as wl  # noqa: E402

METRIC = "k-points/sec (full nbands)"
UNIT = "k-points/s"


def dense_kpath(w: wl.Workload, world: int, rank: int) -> np.ndarray:
    """Rank r's share of the workload's closed k-path sampled world x denser (indices r::world)."""
    if world == 1:
        return w.kpts
    cell = w.cells[0]
    path = wl.SQUARE_PATH if np.allclose(cell.lattice, wl.SQUARE) else wl.HEX_PATH
    return np.ascontiguousarray(wl.kpath(cell.lattice, path, w.nk * world)[rank::world])


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.stop, self.thread = index, [], threading.Event(), None

    def _run(self):
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([x.strip() for x in out.strip().split(",")])
            except Exception:
                pass
            self.stop.wait(0.2)

    def __enter__(self):
        self.thread = threading.Thread(target=self._run, daemon=True)
        self.thread.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.thread.join(timeout=6)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except ValueError:
                continue
            for nme, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------------------------------------ CPU oracle arm
def oracle_sample(w: wl.Workload, kpts: np.ndarray, nsample: int):
    """Times the oracle as it stands on a bounded sample: one assembly + `nsample` k-points spread over the path.
    Returns (extrapolated whole-workload k-points/s, t_assemble, t_per_k, threads used)."""
    import oracle
    cell = w.cells[0]
    t0 = time.perf_counter()
    comp = oracle.isotropic_plane_strain_compliance(cell.E, cell.nu)
    Phi, Psi = oracle.assemble(cell.lattice, cell.vert_offset, cell.verts, comp, cell.rho, w.Mt)
    t_asm = time.perf_counter() - t0
    idx = np.unique(np.linspace(0, len(kpts) - 1, nsample).round().astype(int))
    t0 = time.perf_counter()
    for i in idx:
        oracle.bands_at_k(Phi, Psi, cell.lattice, w.Mt, kpts[i], w.nbands)
    t_k = (time.perf_counter() - t0) / len(idx)
    nk_total = len(kpts) * len(w.cells)
    total = len(w.cells) * t_asm + nk_total * t_k
    try:
        from threadpoolctl import threadpool_info
        threads = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        threads = os.cpu_count() or 1
    return nk_total / total, t_asm, t_k, threads, len(idx)


def oracle_single_thread_seconds(w: wl.Workload, kpts: np.ndarray):
    """One k-point of the oracle with the BLAS pool limited to one thread (the paper's baseline is serial).
    Returns seconds per k-point, or None when threadpoolctl is missing."""
    import oracle
    try:
        from threadpoolctl import threadpool_limits
    except Exception:
        return None
    cell = w.cells[0]
    comp = oracle.isotropic_plane_strain_compliance(cell.E, cell.nu)
    Phi, Psi = oracle.assemble(cell.lattice, cell.vert_offset, cell.verts, comp, cell.rho, w.Mt)
    with threadpool_limits(limits=1):
        t0 = time.perf_counter()
        oracle.bands_at_k(Phi, Psi, cell.lattice, w.Mt, kpts[len(kpts) // 2], w.nbands)
        return time.perf_counter() - t0


def factored_once_seconds(w: wl.Workload, kpts: np.ndarray, nsample: int):
    """A second, fairer CPU figure next to the oracle's (which re-factors Phi at every k-point by design): Phi and Psi
    are Cholesky-factored ONCE, K(k) = (L^-1 H)^H (L^-1 H), and LAPACK returns only the lowest nbands eigenvalues.
    SciPy calls written here, not oracle code.  Returns (seconds of the one-off factorisations, seconds per k-point)."""
    import oracle
    import scipy.linalg as sla
    cell = w.cells[0]
    comp = oracle.isotropic_plane_strain_compliance(cell.E, cell.nu)
    Phi, Psi = oracle.assemble(cell.lattice, cell.vert_offset, cell.verts, comp, cell.rho, w.Mt)
    _, _, V = oracle.reciprocal_basis(cell.lattice)
    t0 = time.perf_counter()
    Lp = np.linalg.cholesky(Phi)
    Ls = np.linalg.cholesky(Psi)
    t_fac = time.perf_counter() - t0
    idx = np.unique(np.linspace(0, len(kpts) - 1, nsample).round().astype(int))
    t0 = time.perf_counter()
    for i in idx:
        H = V * oracle.coupling_B(cell.lattice, w.Mt, kpts[i])
        X = sla.solve_triangular(Lp, H, lower=True)
        W = sla.solve_triangular(Ls, X.conj().T, lower=True).conj().T        # L_Phi^-1 H L_Psi^-H
        sla.eigh(W.conj().T @ W, eigvals_only=True, subset_by_index=[0, w.nbands - 1])
    return t_fac, (time.perf_counter() - t0) / len(idx)


def oracle_nsample(w: wl.Workload) -> int:
    return {"C1": 30, "C2": 12, "C3": 6, "C4": 10, "C5": 3}.get(w.name, 4)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = wl.get(args.workload) if args.workload != "C4" else wl.get("C4", ncells=args.cells)
    ns = oracle_nsample(w)
    vals, t0 = [], time.perf_counter()
    for i in range(args.warmup + args.steps):
        v, t_asm, t_k, threads, nidx = oracle_sample(w, w.kpts, ns)
        if i >= args.warmup:
            vals.append(v)
        if time.perf_counter() - t0 > 240 and vals:      # keep the whole run within a few minutes
            break
    value = float(np.mean(vals))
    sample = (f"per step: 1 assembly (Mt={w.Mt}) + {nidx} of {w.nk} k-points (zhegv, all {2 * w.N} eigenvalues), "
              f"extrapolated to the whole workload ({len(w.cells)} cell(s) x {w.nk} k-points)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": len(vals),
            "warmup": args.warmup, "ms_per_step": 1e3 * w.nk * len(w.cells) / value, "higher_is_better": True,
            # value and ms_per_step are EXTRAPOLATED from the sample below (the oracle is too slow to run whole):
            "extrapolated": True, "nsample_kpoints": int(nidx), "nk_total": int(w.nk * len(w.cells)),
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{w.name}: {w.description}"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------ CUDA arm
HBM_CLASSES = {"hemv", "expand", "pencil", "combine"}
TENSOR_CLASSES = {"gemm_factor", "gemm_reduce", "gemm_tridiag", "gemm_hemm", "gemm_wy"}
# zgemm_kernel executes the 3M complex product: 6 real flops per complex multiply-add of the 8 the algorithm counts
GEMM_EXECUTED_OVER_ALGORITHMIC = 6.0 / 8.0
TABLE_EXECUTED_OVER_ALGORITHMIC = 76.0 / 118.0  # table_sep_kernel (static SASS count per term) vs the direct formula


def measure(bs, torch, w, kpts, steps, warmup, local, barrier, e2e=True):
    """Times `steps` passes of the whole path over workload `w` at the k-points `kpts` on the current device.
    Returns a dict: device-resident pass (ms_total, launches, clocks), the per-kernel pass (kacc, stage_acc) and the
    end-to-end pass from host buffers."""
    nk, ncell = len(kpts), len(w.cells)
    comps = [bs.bs_isotropic_plane_strain(c.E, c.nu) for c in w.cells]

    # cells that share one geometry (config 4: every cell is the same 8 x 8 pixel grid with other materials) are created
    # through bs_create_cells_shared: S1 integrates the polygons once and forms every cell's table as T = W I
    c0 = w.cells[0]
    same_geometry = ncell > 1 and all(np.array_equal(c.lattice, c0.lattice) and np.array_equal(c.vert_offset, c0.vert_offset)
                                      and np.array_equal(c.verts, c0.verts) for c in w.cells)

    def create(timing):
        if same_geometry:
            hs = bs.bs_create_cells_shared(c0.lattice, c0.vert_offset, c0.verts, np.stack(comps), np.stack([c.rho for c in w.cells]))
        else:
            hs = [bs.bs_create_cell(c.lattice, c.vert_offset, c.verts, comp, c.rho) for c, comp in zip(w.cells, comps)]
        bs.bs_set_option(hs[0], bs.BS_OPT_TIMING, timing)
        return hs

    cells = create(0)
    ws_bytes = bs.bs_workspace_bytes(cells[0], w.Mt, nk)
    workspaces = [torch.empty(ws_bytes, dtype=torch.uint8, device="cuda") for _ in cells]
    for h, t in zip(cells, workspaces):
        bs.bs_set_workspace(h, t)
    out_dev = torch.empty(ncell, nk, w.nbands, dtype=torch.float64, device="cuda")
    kacc, stage_acc = {}, np.zeros(bs.BS_T_COUNT)

    def accumulate():
        for k, (ms, work, cnt) in bs.bs_get_kernel_timings(cells[0]).items():
            a = kacc.setdefault(k, [0.0, 0.0, 0])
            a[0] += ms; a[1] += work; a[2] += cnt

    def step(record):
        bs.bs_assemble_batch(cells, w.Mt)
        if record:
            accumulate()
        bs.bs_bands_batch(cells, kpts, w.nbands, out=out_dev)
        if record:
            accumulate()
            stage_acc[:] += bs.bs_get_timings(cells[0])

    for _ in range(max(warmup, 3)):
        step(False)
    # ---- pass 1: the product path as a caller runs it (no per-kernel events, asynchronous on the stream) -> value
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = bs.bs_launch_count(cells[0])
    barrier()
    with ClockSampler(local) as clk:
        e0.record()
        for _ in range(steps):
            step(False)
        e1.record()
        barrier()
    res = {"ms_total": e0.elapsed_time(e1), "launches": bs.bs_launch_count(cells[0]) - l0, "clocks": clk.summary(),
           "ws_bytes": ws_bytes, "nk": nk, "ncell": ncell}
    # ---- pass 2: the same steps again with CUDA events around every launch on the launching stream
    # (BS_OPT_TIMING = 2) -> per-kernel durations for the roofline.  Kept out of pass 1 because two event records per
    # launch and a synchronise per call slow the launch-bound small configs down by up to 20 %.
    bs.bs_set_option(cells[0], bs.BS_OPT_TIMING, 2)
    step(False)
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    p0.record()
    for _ in range(steps):
        step(True)
    p1.record()
    barrier()
    res.update({"ms_profiled": p0.elapsed_time(p1), "kacc": kacc, "stage_acc": stage_acc})
    lam_dev = out_dev.cpu().numpy()
    res["lam"] = lam_dev
    for h in cells:
        bs.bs_destroy_cell(h)
    if not e2e:
        return res
    # ---- end to end through the public API with host buffers (H2D of the geometry, D2H of omega^2 inside the region)
    out_host = np.empty((ncell, nk, w.nbands))

    def e2e_step():
        hs = create(0)
        for h, t in zip(hs, workspaces):
            bs.bs_set_workspace(h, t)
        bs.bs_assemble_batch(hs, w.Mt)
        bs.bs_bands_batch(hs, kpts, w.nbands, out=out_host)
        for h in hs:
            bs.bs_destroy_cell(h)

    for _ in range(max(warmup, 3)):
        e2e_step()
    barrier()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk_e2e:
        f0.record()
        for _ in range(steps):
            e2e_step()
        f1.record()
        barrier()
    assert np.array_equal(out_host, lam_dev), "e2e and device-resident results differ"
    res.update({"ms_e2e": f0.elapsed_time(f1), "clocks_e2e": clk_e2e.summary(), "d2h": out_host.nbytes,
                "h2d": sum(c.lattice.nbytes + c.vert_offset.nbytes + c.verts.nbytes + comp.nbytes + c.rho.nbytes
                           for c, comp in zip(w.cells, comps)) + kpts.nbytes})
    return res


def kernel_groups(kacc):
    """Timing classes grouped by the __global__ function they launch (all DMMA GEMM classes are zgemm_kernel)."""
    groups = {}
    for k, a in kacc.items():
        if not a[2]:
            continue
        gname = "zgemm_kernel" if k in TENSOR_CLASSES else k
        gacc = groups.setdefault(gname, [0.0, 0.0, 0, []])
        gacc[0] += a[0]; gacc[1] += a[1]; gacc[2] += a[2]; gacc[3].append(k)
    return groups


def s6_fraction(bs, w, res, steps, dmma_peak):
    n = 2 * w.N
    tri_ms = res["stage_acc"][bs.BS_T_TRIDIAG]
    tri_flops = 16.0 * n ** 3 / 3.0 * res["nk"] * res["ncell"] * steps
    return (tri_flops / (tri_ms * 1e9) / dmma_peak) if tri_ms else None


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_1310_6380_b200 as bs

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def get_workload(name):
        return wl.get(name) if name != "C4" else wl.get("C4", ncells=args.cells)

    w = get_workload(args.workload)
    kpts = dense_kpath(w, world, rank)
    nk, ncell = len(kpts), len(w.cells)
    dmma_peak, dfma_peak = bs.bs_fp64_peak()
    res = measure(bs, torch, w, kpts, args.steps, args.warmup, local, barrier)
    ms_total, ms_e2e = res["ms_total"], res["ms_e2e"]

    # ---- strong scaling (N > 1): the SAME k-path (or cell batch) split contiguously over the ranks by the sharded driver,
    # replicated assembly, one all-gather of the results; every rank ends up with the whole band structure
    strong = None
    if world > 1:
        from paper_1310_6380_b200 import sharded
        inputs = [(c.lattice, c.vert_offset, c.verts, bs.bs_isotropic_plane_strain(c.E, c.nu), c.rho) for c in w.cells]
        for _ in range(3):
            lam_all = sharded.bands_sharded(inputs, w.Mt, w.kpts, w.nbands)
        barrier()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record()
        for _ in range(args.steps):
            lam_all = sharded.bands_sharded(inputs, w.Mt, w.kpts, w.nbands)
        s1.record()
        barrier()
        ms_strong = s0.elapsed_time(s1)
        t = torch.tensor([ms_total, ms_e2e, ms_strong], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total, ms_e2e, ms_strong = float(t[0]), float(t[1]), float(t[2])
        strong = {"value": w.nk * ncell * args.steps / (ms_strong * 1e-3), "unit": UNIT, "ms_per_step": ms_strong / args.steps,
                  "what": "the workload's own k-path split contiguously over the ranks (paper_1310_6380_b200.sharded), "
                          "assembly replicated, all-gather of nk x nbands doubles; handles created and destroyed per step",
                  "axis": sharded.choose_axis(ncell, w.nk, world)}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    units = nk * ncell * world * args.steps
    value = units / (ms_total * 1e-3)
    hbm_peak, hbm_src = measured_peaks()
    # ---- roofline of the dominant KERNEL: the kernel with the largest share of device time inside the timed region.
    # Every kernel's own figures are listed under "by_kernel".
    kacc = res["kacc"]
    tot_kernel_ms = sum(a[0] for a in kacc.values()) or 1.0
    groups = kernel_groups(kacc)
    tjson, tsrc = {}, None
    tpath = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if os.path.exists(tpath):
        tall = json.load(open(tpath))
        tjson, tsrc = tall.get(w.name, {}), tall.get("_source")

    def roof_of(gname):
        ms_d, work_d, cnt_d, classes = groups[gname]
        if gname == "zgemm_kernel":
            r = {"bound": "tensor", "achieved": work_d / (ms_d * 1e9), "peak": dmma_peak, "unit": "TFLOP/s",
                 "peak_source": "FP64 DMMA (mma.sync m8n8k4) register-only loop measured in this run by bs_fp64_peak; "
                                "MEASURED_PEAKS.json has no FP64 entry"}
            # the kernel EXECUTES the 3M product (6 of the 8 algorithmic flops per complex multiply-add): this is how
            # busy the DMMA pipe really is, i.e. the headroom left in the kernel
            r["achieved_executed"] = r["achieved"] * GEMM_EXECUTED_OVER_ALGORITHMIC
            r["frac_executed"] = r["achieved_executed"] / dmma_peak
        elif gname in HBM_CLASSES:
            r = {"bound": "hbm", "achieved": work_d / (ms_d * 1e6), "peak": hbm_peak, "unit": "GB/s", "peak_source": hbm_src}
        else:
            r = {"bound": "alu", "achieved": work_d / (ms_d * 1e9) if work_d else None, "peak": dfma_peak,
                 "unit": "TFLOP/s", "peak_source": "FP64 DFMA register-only loop measured in this run by bs_fp64_peak"}
        r["frac"] = (r["achieved"] / r["peak"]) if r["achieved"] else None
        if gname == "table" and r["achieved"]:
            # S1's algorithmic count is the directly evaluated formula (sincospi + sinpi + 14 channel FMAs = 118 flops
            # per (index difference, edge) term by the SASS of the direct kernel); the separable-phase kernel executes
            # at most 76 (static SASS count, profiles/r2_s1_table.md), so its FP64 pipe is at most this busy:
            r["achieved_executed"] = r["achieved"] * TABLE_EXECUTED_OVER_ALGORITHMIC
            r["frac_executed"] = r["achieved_executed"] / r["peak"]
        if r["bound"] == "hbm" and r["frac"] and r["frac"] > 1.0:
            r["note"] = ("algorithmic bytes / time exceeds the HBM copy peak: part of the operands is served by L2 "
                         "(small per-cell matrices reused across the k-points of the launch)")
        r.update({"kernel": gname, "classes": sorted(classes), "launches_per_step": cnt_d / args.steps,
                  "avg_launch_ms": ms_d / max(cnt_d, 1), "share_of_kernel_time": ms_d / tot_kernel_ms,
                  "traffic": tjson.get(gname), "work_per_launch": work_d / max(cnt_d, 1)})
        if tjson.get(gname) is not None:
            r["traffic_source"] = tsrc      # a committed ncu capture, not a measurement of this run
        return r

    dom = max(groups, key=lambda k: groups[k][0])
    roof = roof_of(dom)
    roof["measured_in"] = ("second pass of the same %d steps with CUDA events around every launch (BS_OPT_TIMING = 2), "
                           "%.3f ms per step; value comes from the first pass without them" % (args.steps, res["ms_profiled"] / args.steps))
    roof["by_kernel"] = [{k: v for k, v in roof_of(gname).items() if k != "peak_source"}
                         for gname in sorted(groups, key=lambda k: -groups[k][0])]
    n = 2 * w.N
    gemm_ms = sum(kacc[k][0] for k in TENSOR_CLASSES if k in kacc)
    gemm_fl = sum(kacc[k][1] for k in TENSOR_CLASSES if k in kacc)
    stage_acc = res["stage_acc"]
    tri_ms = stage_acc[bs.BS_T_TRIDIAG]
    tri_flops = 16.0 * n ** 3 / 3.0 * nk * ncell * args.steps
    stages = {nme: stage_acc[i] / args.steps for i, nme in
              enumerate(["table_ms", "expand_ms", "factor_ms", "coef_ms", "pencil_ms", "tridiag_ms", "bisect_ms"])}
    stages["kernels"] = {k: {"ms_per_step": a[0] / args.steps, "launches_per_step": a[2] / args.steps}
                         for k, a in kacc.items() if a[2]}
    stages["fp64_tensor"] = {"all_dmma_gemm_tflops": gemm_fl / (gemm_ms * 1e9) if gemm_ms else None,
                             "tridiag_algorithmic_tflops": tri_flops / (tri_ms * 1e9) if tri_ms else None,
                             "tridiag_frac_of_dmma_peak": tri_flops / (tri_ms * 1e9) / dmma_peak if tri_ms else None,
                             "dmma_peak_tflops": dmma_peak, "dfma_peak_tflops": dfma_peak}
    # ---- the other configs, a few steps each (N = 1, default workload only), so that every row of BASELINE.md's table is
    # measured by the same run
    all_configs = None
    if world == 1 and args.workload == "C5" and not args.no_all:
        all_configs = {}
        for name in ("C1", "C2", "C3", "C4"):
            wo = get_workload(name)
            ro = measure(bs, torch, wo, wo.kpts, 5, 3, local, barrier)
            go = kernel_groups(ro["kacc"])
            do = max(go, key=lambda k: go[k][0])
            uo = wo.nk * len(wo.cells) * 5
            all_configs[name] = {"workload": wo.description, "value": uo / (ro["ms_total"] * 1e-3), "unit": UNIT,
                                 "ms_per_step": ro["ms_total"] / 5, "e2e": uo / (ro["ms_e2e"] * 1e-3), "steps": 5,
                                 "s6_frac_of_dmma": s6_fraction(bs, wo, ro, 5, dmma_peak), "dominant_kernel": do,
                                 "dominant_share": go[do][0] / (sum(g[0] for g in go.values()) or 1.0),
                                 "gpu_launches": int(ro["launches"])}
        all_configs["C5"] = {"workload": w.description, "value": value, "unit": UNIT, "ms_per_step": ms_total / args.steps,
                             "e2e": units / (ms_e2e * 1e-3), "steps": args.steps,
                             "s6_frac_of_dmma": stages["fp64_tensor"]["tridiag_frac_of_dmma_peak"], "dominant_kernel": dom,
                             "dominant_share": roof["share_of_kernel_time"], "gpu_launches": int(res["launches"])}
    # ---- CPU oracle on a bounded sample, rank 0, N = 1 only
    cpu = None
    if world == 1 and not args.no_cpu:
        v, t_asm, t_k, threads, nidx = oracle_sample(w, kpts, oracle_nsample(w))
        t1 = oracle_single_thread_seconds(w, kpts)
        t_fac, t_kf = factored_once_seconds(w, kpts, oracle_nsample(w))
        cpu = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "single_thread_s_per_kpoint": t1,
               "extrapolated": True, "nsample_kpoints": int(nidx),
               "sample": f"1 assembly ({t_asm:.2f} s) + {nidx} of {nk} k-points ({t_k:.3f} s each, zhegv all "
                         f"{n} eigenvalues), extrapolated to {ncell} cell(s) x {nk} k-points",
               # the oracle re-solves with Phi at every k-point (it is a checker, not a fast program); a CPU program that
               # factors Phi and Psi once and asks LAPACK for the lowest nbands only is this much faster:
               "factored_once": {"value": ncell * nk / (ncell * (t_asm + t_fac) + ncell * nk * t_kf), "unit": UNIT,
                                 "s_per_kpoint": t_kf, "s_factorisations": t_fac}}
    ws_bytes = res["ws_bytes"]
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_total / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{w.name}: {w.description}", "kpoints_per_gpu": nk, "cells": ncell,
                       "band_structure_wall_ms": ms_total / args.steps,
                       "l2": f"inputs larger than L2: the per-step working set ({ncell * ws_bytes / 2**20:.0f} MiB workspace) "
                             "exceeds the 126 MB L2" if ncell * ws_bytes > 2 * 126e6 else
                             "working set fits L2 (small config): latency-bound, the roofline fraction is not meaningful"},
            "clocks": res["clocks"],
            "e2e": {"value": units / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(res["h2d"]),
                    "d2h_bytes_per_step": int(res["d2h"]), "clocks": res["clocks_e2e"]},
            "gpu_launches": int(res["launches"]), "roofline": roof, "cpu_baseline": cpu, "stages": stages}
    if strong is not None:
        line["strong"] = strong
    if all_configs is not None:
        line["all_configs"] = all_configs
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C5", choices=list(wl.CONFIGS))
    ap.add_argument("--cells", type=int, default=256, help="number of cells of workload C4")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-all", action="store_true", help="skip the short runs of C1-C4 after the default workload")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
