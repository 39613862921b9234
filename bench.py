#!/usr/bin/env python
"""bench.py -- throughput of the fused Chebyshev-filter H~X path on the BASELINE.json workloads.

A "step" is one cheb_filter call (m fused operator steps: gather -> cell contraction -> scatter + recurrence) on one block
of B vectors (config 5: its 200 shifted applies).  metric = GDoF-vectors/s = N_free * B * m * steps / time (reading R14).
Rank 0 prints ONE JSON line.  The line's `value` is the largest single-GPU workload (config 4); `workloads` carries the
same measurement (value, roofline, clocks) for the other roofline workloads 2, 3 and 5; `peaks` the step-0 ceilings
measured in the same run (fe_diag_peak).  See DESIGN.md "Measurement" for the roofline arithmetic.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 2|3|4|5] [--also 2,3,5] [--orders] [--consumers]
                  [--scaling weak|strong] [--impl reference] [--stub]
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "FE H~X GDoF-vectors/s (FP64) in Chebyshev filter"
UNIT = "GDoF-vectors/s"
# nominal FP64 ALU peak: 148 SMs x 64 DFMA/clk/SM x 2 flop x 1.965 GHz (MEASURED_PEAKS.json sm_max_mhz)
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12

# dram__bytes_read.sum + dram__bytes_write.sum of ONE k_apply_tma launch, copied from the committed `ncu --set full`
# captures named here (profiles/); not measured in this run
NCU_TRAFFIC = {
    2: (296.26e6 + 219.88e6, "profiles/r2_c2_k_apply_tma_full.md"),
    3: (3.4587e9 + 3.1621e9, "profiles/r2_c3_k_apply_tma_full.md"),
    4: (35.660e9 + 31.926e9, "profiles/r2_c4_k_apply_tma_full.md"),
    5: (296.34e6 + 97.02e6, "profiles/r2_c5_k_apply_tma_full.md (the kernel alone; the zero-fill of Y writes 141 MB more)"),
}


def algorithmic_flops_per_cell_vector(p):
    """matrix-free sum factorisation in the generic 12-sweep form, 24 n^4 + 9 n^3 flops per cell-vector."""
    n = p + 1
    return 24 * n**4 + 9 * n**3


def executed_fp64_per_cell_vector(p):
    """What k_apply_tma executes per cell-vector (counted from the kernel's structure, cross-checked against the ncu opcode
    mix in profiles/): 10 even-odd sweeps of n^2 lines -- a line costs n DMUL, c h + h (h-1) DFMA and 4 h DADD with
    h = n // 2, c = (n + 1) // 2 -- plus 2 DMUL + 3 DFMA per point (scalings, V, the two geometry ratios).
    Returns (instructions, flops)."""
    n = p + 1
    h, c = n // 2, (n + 1) // 2
    mul, fma, add = n, c * h + h * (h - 1), 4 * h
    lines = 10 * n * n
    instr = lines * (mul + fma + add) + 5 * n**3
    flops = lines * (mul + add + 2 * fma) + (2 + 2 * 3) * n**3
    return instr, flops


def spectrum_bounds(w):
    """Filter window for the timed runs.  Bounds only steer values, not work: b from the kinetic-only estimate
    3*mu_max^2*alpha_max of SURVEY 8(c) is replaced by a safe closed-form over-estimate, a0 below the deepest well."""
    hmin = min(np.diff(w.xe).min(), np.diff(w.ye).min(), np.diff(w.ze).min())
    b = 3.0 * (2.0 * w.p * w.p / hmin) ** 2 * 0.5 + 10.0
    R, Z = (np.zeros((1, 3)), np.array([0.0])) if w.potential == "harmonic" else w.atom_list()
    a0 = -2.0 * float(Z.sum()) - 1.0
    return a0, a0 + 0.05 * (b - a0), b


class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.FIELDS,
                                       "--format=csv,noheader,nounits", "-lms", "50"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            parts = [s.strip() for s in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
                pw.append(float(parts[2]))
            except ValueError:
                continue
            for nme, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nme)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm),
                       power_w_max=float(max(pw)) if pw else None)
        return out


# ---- the oracle on the host cores (cpu_baseline leg and --impl reference) -------------------------------------------------
def cpu_baseline(w_index, sample, steps=1, all_cores=True):
    """The oracle as it stands, on a bounded sample: the same recipe on a centred sub-mesh of budget_cells^3 cells, the
    first ncols columns of the block (columns are independent, R22), full degree m (config 5: 4 shifted applies).
    Setup (cell matrices, CSR) is not timed."""
    import oracle
    budget_cells, ncols = sample
    w = workloads.reduced(w_index, budget_cells)
    w.B = min(w.B, ncols)
    om = oracle.OracleMesh(w.xe, w.ye, w.ze, w.p)
    om.set_potential(w.V(om.quad_coords()))
    om.assemble()
    mask = om.mask()
    X = workloads.random_block(w.x_seed, om.N, w.B, mask)
    a0, a, b = spectrum_bounds(w)
    napply = w.m if w.m > 0 else 4
    eps = w.eps()

    def run(nthreads):
        t0 = time.perf_counter()
        for _ in range(steps):
            if w.m > 0:
                om.filter(X, w.m, a, b, a0, nthreads=nthreads)
            else:
                for _ in range(napply):
                    om.apply(X, eps, nthreads=nthreads)
        return (time.perf_counter() - t0) / steps

    t1 = run(1)
    out = {"value": om.N_free * w.B * napply / t1 / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
           "sample": "%s: centred %d^3-cell sub-mesh (N=%d), %d columns, %d applies, serial CSR oracle; setup untimed"
                     % (w.name, budget_cells, om.N, w.B, napply),
           "seconds_per_step": t1}
    if all_cores:
        nc = os.cpu_count() or 1
        tn = run(nc)
        out["value_all_cores"] = om.N_free * w.B * napply / tn / 1e9
        out["cores_all"] = nc
    return out


SAMPLE_CELLS = {2: (6, 64), 3: (4, 8), 4: (4, 8), 5: (6, 64)}  # (cells per axis, columns) of the oracle's timed sample


def run_reference(args):
    """--impl reference: the oracle timed on the host cores, same metric / config; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = workloads.config(args.workload)
    for _ in range(min(args.warmup, 1)):
        cpu_baseline(args.workload, (2, 2), 1, all_cores=False)
    cb = cpu_baseline(args.workload, SAMPLE_CELLS[args.workload], max(1, args.steps), all_cores=False)
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": cb["seconds_per_step"] * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.describe(), "sample": cb["sample"]},
            "cpu_baseline": {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ---- rank plumbing (one process per GPU; columns are sharded with no exchange) --------------------------------------------
def respawn_under_torchrun(args):
    """`python bench.py --gpus N` without a torchrun environment: start N ranks of this script on this node."""
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def columns_of_rank(w, rank, world, scaling):
    """weak: every rank filters its own B-column block; strong: the B columns of the workload are dealt to the ranks."""
    from paper_2510_10529_b200.colsplit import column_slice
    if scaling == "weak":
        return w.B
    lo, hi = column_slice(w.B, rank, world)
    return hi - lo


def job_line(w, per_rank, world, dist, device, steps, warmup, scaling):
    """Whole-job numbers from the per-rank measurement: times are the max over ranks, units the sum over ranks."""
    from paper_2510_10529_b200.colsplit import job_throughput, max_over_ranks
    ms_step, e2e_ms = max_over_ranks([per_rank["ms_per_step"], per_rank.get("e2e_ms_per_step", 0.0)], dist, device)
    cols = per_rank["B"] * world if scaling == "weak" else w.B
    units = per_rank["N_free"] * cols * per_rank["napply"]  # DoF-vectors per step, all ranks
    value = job_throughput(units / world, world, ms_step * 1e-3) / 1e9
    e2e = job_throughput(units / world, world, e2e_ms * 1e-3) / 1e9 if e2e_ms > 0 else None
    return {"value": value, "ms_per_step": ms_step, "e2e_value": e2e, "e2e_ms_per_step": e2e_ms, "n_gpus": world,
            "steps": steps, "warmup": warmup, "scaling": scaling, "columns_total": cols}


def stub_measurement(w, rank, B):
    """--stub: no GPU work; a fixed fake step time per rank, so that the spawning, the barrier, the max over ranks and the
    whole-job aggregation can be exercised on CPU (gloo).  The line says "data": "stub"."""
    return {"ms_per_step": 10.0 * (1 + rank), "e2e_ms_per_step": 20.0 * (1 + rank), "napply": max(w.m, 1), "N": w.N,
            "N_free": w.N_free, "B": B, "ncells": w.ncells, "launches": 0, "clocks": None, "e2e_bytes": 0}


# ---- device timing --------------------------------------------------------------------------------------------------------
def time_workload(fe, torch, w, B, steps, warmup, dev, seed_offset=0, with_e2e=False, dist=None, variant=0, chain=False):
    """Device-resident timing of `steps` cheb_filter calls (config 5: blocks of 200 shifted applies), CUDA events on the
    launching stream around every step; clocks sampled during the timed region."""
    gm = fe.FEMesh(w.xe, w.ye, w.ze, w.p, device=dev)
    if variant:
        gm.set_variant(variant)
    Vq = w.V(gm.quad_coords())
    gm.set_potential(Vq)
    mask = torch.as_tensor(gm.mask().astype(np.float64), device="cuda")[:, None]
    N = gm.N
    nrot = 3 if N * B * 8 < 1 << 30 else 1  # rotate buffer sets when one block is L2-scale (config 2/5)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(1234 + w.x_seed + seed_offset)
    pristine = torch.randn(N, B, dtype=torch.float64, device="cuda", generator=gen)
    pristine.mul_(mask)
    Xs = [torch.empty_like(pristine) for _ in range(nrot)]
    works = [torch.empty(2 * N * B, dtype=torch.float64, device="cuda") for _ in range(nrot)]
    a0, a, b = spectrum_bounds(w)
    eps = torch.as_tensor(w.eps()[:B], device="cuda") if w.eps_seed is not None else None
    napply = w.m if w.m > 0 else w.n_applies

    def one_step(i):
        X, wk = Xs[i % nrot], works[i % nrot]
        if w.m > 0:
            gm.cheb_filter(X, w.m, a, b, a0, wk)
        else:  # R19: alternate two input and two output blocks
            Y0, Y1 = wk[:N * B].view(N, B), wk[N * B:].view(N, B)
            for t in range(w.n_applies):
                if chain:  # the zero-fill of the next output block rides on this launch (fe_apply_H_chain)
                    gm.apply_H_chain(X if t % 2 == 0 else pristine, Y0 if t % 2 == 0 else Y1, Y1 if t % 2 == 0 else Y0, eps,
                                     y_is_clear=(t > 0))
                else:
                    gm.apply_H(X if t % 2 == 0 else pristine, Y0 if t % 2 == 0 else Y1, eps)

    def restore(i):  # only the block the coming step filters
        Xs[i % nrot].copy_(pristine)

    for i in range(warmup):
        restore(i)
        one_step(i)
    torch.cuda.synchronize()
    sampler = ClockSampler(dev)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    l0 = gm.launches
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    for i in range(steps):
        restore(i)  # outside the timed events
        ev[i][0].record()
        one_step(i)
        ev[i][1].record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    clocks = sampler.stop()
    ms = [e0.elapsed_time(e1) for e0, e1 in ev]
    res = {"ms_per_step": float(sum(ms)) / steps, "ms_min": float(min(ms)), "launches": gm.launches - l0,
           "napply": napply, "N": N, "N_free": gm.N_free, "B": B, "clocks": clocks, "ncells": gm.ncells,
           "l2": ("%d rotating buffer sets of 3 x %.0f MB blocks > 126 MB L2" % (nrot, N * B * 8 / 1e6)) if nrot > 1
                 else "blocks of %.2f GB >> L2" % (N * B * 8 / 1e9)}
    if with_e2e:
        # end to end through the public API with HOST buffers, every step: pinned H2D of the block, the filter, D2H of
        # the result (config 2-4: the C-ABI host call cheb_filter_host; config 5: copies around the 200 applies)
        host_io = torch.empty(N, B, dtype=torch.float64, pin_memory=True)
        host_io.copy_(pristine)
        X, wk = Xs[0], works[0]
        if w.m > 0:  # the host call owns its device staging: release this function's blocks first
            Xs.clear()
            works.clear()
            X = wk = None
            torch.cuda.empty_cache()

        def e2e_step():
            if w.m > 0:
                gm.cheb_filter_host(host_io, w.m, a, b, a0)  # synchronous
            else:
                X.copy_(host_io, non_blocking=True)
                one_step(0)
                host_io.copy_(wk[:N * B].view(N, B), non_blocking=True)
                torch.cuda.synchronize()

        e2e_step()
        host_io.copy_(pristine)
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            e2e_step()
        torch.cuda.synchronize()
        res["e2e_ms_per_step"] = (time.perf_counter() - t0) / steps * 1e3
        res["e2e_bytes"] = N * B * 8
    gm.close()
    return res


def roofline_block(w, r, ms_step, peaks, hbm_peak):
    """The dominant kernel of the step is k_apply_tma (98-99 % of the step: profiles/*launches*): one launch = step / m."""
    flops_launch = algorithmic_flops_per_cell_vector(w.p) * r["ncells"] * r["B"]
    dur = ms_step * 1e-3 / r["napply"]
    ach = flops_launch / dur / 1e12
    instr_cv, flops_cv = executed_fp64_per_cell_vector(w.p)
    peak = max((peaks or {}).get("dfma_tflops") or 0.0, (peaks or {}).get("dmma_tflops") or 0.0) or FP64_NOMINAL_TFLOPS
    ck = r.get("clocks") or {}
    alg_bytes = (24 if w.m > 0 else 16) * r["N"] * r["B"]
    traffic = NCU_TRAFFIC.get(w.index)
    out = {"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
           "peak_source": ("measured in this run: the better of fe_diag_peak kind 0 (register-resident DFMA chains) and kind 1 "
                           "(mma.sync.m8n8k4.f64 chains), best launch -- the two share the FP64 pipe"
                           if (peaks or {}).get("dfma_tflops") else "nominal (no --peaks leg in this run)"),
           "peak_nominal": FP64_NOMINAL_TFLOPS, "frac_of_nominal": ach / FP64_NOMINAL_TFLOPS,
           "frac_kind": "useful work: ALGORITHMIC flops (24 n^4 + 9 n^3 per cell-vector, SURVEY 8(d)) / duration / peak; "
                        "the even-odd kernel EXECUTES fewer flops (executed_*), so 1.0 is not the ceiling of this number",
           "executed_tflops": flops_cv * r["ncells"] * r["B"] / dur / 1e12,
           "executed_over_algorithmic_flops": flops_cv / algorithmic_flops_per_cell_vector(w.p),
           "kernel": "k_apply_tma<p=%d> (one fused operator step: step time / m, CUDA events on the launching stream)" % w.p,
           "launch_ms": dur * 1e3, "algorithmic_bytes": alg_bytes,
           "traffic": traffic[0] if traffic else None,
           "traffic_source": ("committed ncu capture %s (not measured in this run)" % traffic[1]) if traffic else None,
           "hbm_frac_of_measured": (alg_bytes / dur / 1e9 / hbm_peak) if hbm_peak else None}
    if ck.get("sm_mhz"):
        # share of the FP64 pipe's issue cycles the executed instruction count needs at the sampled clock (the number ncu
        # reports as sm__pipe_fp64_cycles_active: a warp-wide FP64 instruction holds a sub-partition's pipe for 2 cycles)
        warp_instr = instr_cv * r["ncells"] * r["B"] / 32.0
        out["fp64_pipe_busy_est"] = warp_instr * 2.0 / (148 * 4 * dur * ck["sm_mhz"] * 1e6)
        if ck.get("sm_max_mhz"):
            out["frac_at_sampled_clock"] = out["frac_of_nominal"] * ck["sm_max_mhz"] / ck["sm_mhz"]
    return out


def measure_peaks(fe, dev):
    """Step-0 ceilings, measured through the C ABI (fe_diag_peak) before the timed workloads."""
    sampler = ClockSampler(dev)
    out = {"dfma_tflops": fe.fe_diag_peak(0, 0.4, dev), "dmma_tflops": fe.fe_diag_peak(1, 0.4, dev),
           "stream_2r1w_gbs": fe.fe_diag_peak(2, 0.3, dev), "bulk_reduce_add_gbs": fe.fe_diag_peak(3, 0.3, dev),
           "red_global_add_gbs": fe.fe_diag_peak(4, 0.3, dev)}
    out["clocks"] = sampler.stop()
    out["how"] = ("fe_diag_peak: best launch of >= 0.3 s back to back; DFMA = 8 chains x 8 warps x 4 CTAs/SM; DMMA = "
                  "mma.sync.m8n8k4.f64 chains; stream = y = a x + z on 1 GiB arrays (3 x 8 B per element); reduce-add = "
                  "payload bytes of cp.reduce.async.bulk.add.f64 / red.global.add.f64 into a 1 GiB array")
    return out


GBOX_TRAFFIC = 1.072e9 + 0.900e9  # ncu DRAM read + write of one k_apply_gbox launch on the adaptive workload (profiles/r2b_gbox_*)


def time_adaptive(fe, torch, dev, peaks, hbm_peak, steps, warmup, p=6, B=64, m=30, generic=False):
    """NEXT-3 workload (not a BASELINE.json config): config 3's atoms on an adaptively refined mesh with hanging nodes
    (workloads.adaptive_molecule: 12^3 root cells refined twice around the nuclei), cheb_filter of degree m through the
    general-mesh path (explicit l2g, constraint expansion / collapse).  The leaves are axis-aligned boxes, so the default is
    the 10-sweep box-cell kernel of fe_gbox.cuh; generic=True (fe_set_variant 9) times the 12-sweep kernel with a full 3 x 3
    metric (fe_general.cuh) that deformed cells need, on the same mesh.  The roofline uses the algorithmic count
    24 n^4 + 9 n^3 per cell-vector of SURVEY 8(d) for both."""
    mesh, V = workloads.adaptive_molecule()
    gm = fe.FEMesh.general(mesh, p, device=dev)
    if generic:
        gm.set_variant(9)
    gm.set_potential(V(gm.quad_coords()))
    N = gm.N
    gen = torch.Generator(device="cuda")
    gen.manual_seed(4321)
    mask = torch.as_tensor(gm.mask().astype(np.float64), device="cuda")[:, None]
    pristine = torch.randn(N, B, dtype=torch.float64, device="cuda", generator=gen) * mask
    X = torch.empty_like(pristine)
    work = torch.empty(2 * N * B, dtype=torch.float64, device="cuda")
    a0, a, b = -40.0, 20.0, 3.0 * (2.0 * p * p / 0.5) ** 2 * 0.5 + 10.0  # steers values only
    for _ in range(warmup):
        X.copy_(pristine)
        gm.cheb_filter(X, m, a, b, a0, work)
    torch.cuda.synchronize()
    sampler = ClockSampler(dev)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    l0 = gm.launches
    for i in range(steps):
        X.copy_(pristine)
        ev[i][0].record()
        gm.cheb_filter(X, m, a, b, a0, work)
        ev[i][1].record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = float(sum(e0.elapsed_time(e1) for e0, e1 in ev)) / steps
    dur = ms * 1e-3 / m
    n = p + 1
    flops = algorithmic_flops_per_cell_vector(p) * gm.ncells * B
    peak = max((peaks or {}).get("dfma_tflops") or 0.0, (peaks or {}).get("dmma_tflops") or 0.0) or FP64_NOMINAL_TFLOPS
    alg_bytes = 24 * N * B
    out = {"workload": "adaptive molecule: %d leaves (levels %s) p=%d N=%d unconstrained + %d hanging nodes B=%d m=%d"
                       % (gm.ncells, np.bincount(mesh.cells[:, 0]).tolist(), p, N, gm.N_all - N, B, m),
           "value": gm.N_free * B * m / (ms * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": ms,
           "roofline": {"bound": "alu", "achieved": flops / dur / 1e12, "peak": peak, "unit": "TFLOP/s",
                        "frac": flops / dur / 1e12 / peak, "frac_of_nominal": flops / dur / 1e12 / FP64_NOMINAL_TFLOPS,
                        "kernel": "%s<p=%d> + k_gen_init / k_gen_expand / k_gen_collapse (one operator step: step / m)"
                                  % ("k_apply_gen" if generic else "k_apply_gbox", p),
                        "launch_ms": dur * 1e3, "algorithmic_bytes": alg_bytes,
                        "traffic": (1.101e9 + 0.469e9) if generic else GBOX_TRAFFIC,
                        "traffic_source": "committed ncu capture profiles/%s (the cell kernel alone, not measured in this run)"
                                          % ("r2_general_k_apply_gen.md" if generic else "r2b_gbox_k_apply_gbox.md"),
                        "hbm_frac_of_measured": (alg_bytes / dur / 1e9 / hbm_peak) if hbm_peak else None},
           "clocks": clocks, "gpu_launches": int(gm.launches - l0)}
    gm.close()
    return out


def time_orders(fe, torch, dev, peaks, hbm_peak, steps, warmup):
    """--orders: every Lagrange order p = 2..8 on one ~2 M-node uniform mesh (B = 64, degree-12 filter, the config-2 well),
    default launch shapes: the table of DESIGN.md 6.2."""
    out = {}
    for p in range(2, 9):
        cells = max(2, int(round((2.0e6 ** (1.0 / 3.0) - 1) / p)))
        e = workloads.uniform_edges(-10.0, 10.0, cells)
        w = workloads.Workload(20 + p, "orders-p%d" % p, (e, e, e), p, 64, 12, "single", x_seed=20 + p)
        r = time_workload(fe, torch, w, w.B, steps, warmup, dev)
        rf = roofline_block(w, r, r["ms_per_step"], peaks, hbm_peak)
        out["p%d" % p] = {"cells": cells, "N": r["N"], "ms_per_apply": r["ms_per_step"] / w.m,
                          "value": r["N_free"] * w.B * w.m / (r["ms_per_step"] * 1e-3) / 1e9, "unit": UNIT,
                          "frac": rf["frac"], "frac_of_nominal": rf["frac_of_nominal"],
                          "fp64_pipe_busy_est": rf.get("fp64_pipe_busy_est"), "sm_mhz": (r["clocks"] or {}).get("sm_mhz")}
        torch.cuda.empty_cache()
    return out


def time_consumers(fe, torch, w, dev):
    """--consumers: NEXT-1 / NEXT-2 on the workload's mesh (informational): one Rayleigh-Ritz call on a filtered block,
    the Gram product alone, and a fixed number of preconditioned MINRES steps with the config-5 shifts."""
    gm = fe.FEMesh(w.xe, w.ye, w.ze, w.p, device=dev)
    gm.set_potential(w.V(gm.quad_coords()))
    N, B = gm.N, w.B
    gen = torch.Generator(device="cuda")
    gen.manual_seed(99)
    mask = torch.as_tensor(gm.mask().astype(np.float64), device="cuda")[:, None]
    X = torch.randn(N, B, dtype=torch.float64, device="cuda", generator=gen) * mask
    a0, a, b = spectrum_bounds(w)
    gm.cheb_filter(X, 4, a, b, a0)
    work = torch.empty(N * B, dtype=torch.float64, device="cuda")
    Y = X.clone()
    gm.rayleigh_ritz(Y, work)  # warm-up
    Y.copy_(X)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    gm.rayleigh_ritz(Y, work)
    torch.cuda.synchronize()
    rr_ms = (time.perf_counter() - t0) * 1e3
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(10):
        gm.gram(X, Y)
    e1.record()
    torch.cuda.synchronize()
    gram_ms = e0.elapsed_time(e1) / 10
    eps = torch.as_tensor(workloads.shifts(2005, B), device="cuda")
    G = torch.randn(N, B, dtype=torch.float64, device="cuda", generator=gen) * mask
    gm.minres_shifted(G, eps, maxit=8, tol=0.0)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    _, _, it = gm.minres_shifted(G, eps, maxit=48, tol=0.0)
    torch.cuda.synchronize()
    mr_ms = (time.perf_counter() - t0) * 1e3 / it
    gm.close()
    return {"mesh": w.describe(), "rayleigh_ritz_ms": rr_ms, "gram_ms": gram_ms,
            "gram_tflops": 2.0 * N * B * B / (gram_ms * 1e-3) / 1e12, "gram_gbs": 16.0 * N * B / (gram_ms * 1e-3) / 1e9,
            "minres_ms_per_step": mr_ms, "minres_steps_timed": it}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", type=int, default=4, choices=[2, 3, 4, 5],
                    help="the workload of the line's `value` (default: config 4, the largest single-GPU one)")
    ap.add_argument("--also", default="2,3,5", help="other roofline workloads measured into `workloads` ('' = none)")
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"])
    ap.add_argument("--orders", action="store_true", help="also time p = 2..8 on one ~2 M-node mesh (DESIGN.md 6.2)")
    ap.add_argument("--consumers", action="store_true", help="also time Rayleigh-Ritz / Gram / MINRES on config 2's mesh")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-peaks", action="store_true")
    ap.add_argument("--no-adaptive", action="store_true", help="skip the hanging-node workload (NEXT-3) in `workloads`")
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--stub", action="store_true", help="rank-plumbing self-test on CPU (gloo): no GPU work, fake step times")
    args = ap.parse_args()
    if args.warmup < 3 and not args.stub and args.impl == "native":
        args.warmup = 3  # timing rule: at least three warm-up steps
    if args.impl == "reference":
        run_reference(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        respawn_under_torchrun(args)

    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    w = workloads.config(args.workload)
    B = columns_of_rank(w, rank, world, args.scaling)
    dist = None
    if args.stub:
        device = "cpu"
        if world > 1:
            import torch.distributed as dist
            dist.init_process_group("gloo")
            dist.barrier()
        r = stub_measurement(w, rank, B)
        fe = peaks = hbm_peak = None
    else:
        import paper_2510_10529_b200 as fe
        fe.load_library()  # fails loudly if the CUDA extension is missing
        if not torch.cuda.is_available():
            raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
        device = "cuda"
        if world > 1:
            import torch.distributed as dist
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        torch.cuda.set_device(local)
        hbm_peak = None
        try:
            with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
                hbm_peak = json.load(f)["hbm_gbs"]
        except Exception:
            pass
        peaks = None if args.no_peaks else measure_peaks(fe, local)
        r = time_workload(fe, torch, w, B, args.steps, args.warmup, local, seed_offset=rank, with_e2e=True, dist=dist,
                          variant=args.variant)
    job = job_line(w, r, world, dist, device, args.steps, args.warmup, args.scaling)
    others = {}
    if not args.stub:
        torch.cuda.empty_cache()
        for idx in [int(s) for s in args.also.split(",") if s.strip()]:
            if idx == args.workload:
                continue
            wi = workloads.config(idx)
            Bi = columns_of_rank(wi, rank, world, args.scaling)
            ri = time_workload(fe, torch, wi, Bi, args.steps, args.warmup, local, seed_offset=rank, dist=dist,
                               variant=args.variant)
            ji = job_line(wi, ri, world, dist, device, args.steps, args.warmup, args.scaling)
            others["cfg%d" % idx] = {"workload": wi.describe(), "value": ji["value"], "unit": UNIT,
                                     "ms_per_step": ji["ms_per_step"], "l2": ri["l2"],
                                     "filtered_blocks_per_s": world / (ji["ms_per_step"] * 1e-3) if wi.m > 0 else None,
                                     "roofline": roofline_block(wi, ri, ji["ms_per_step"], peaks, hbm_peak),
                                     "clocks": ri["clocks"], "gpu_launches": int(ri["launches"])}
            if idx == 5:  # the same 200 applies as a chain: every call clears the next call's output block
                rc5 = time_workload(fe, torch, wi, Bi, args.steps, args.warmup, local, seed_offset=rank, dist=dist,
                                    variant=args.variant, chain=True)
                jc5 = job_line(wi, rc5, world, dist, device, args.steps, args.warmup, args.scaling)
                others["cfg5_chain"] = {"workload": wi.describe() + " through fe_apply_H_chain", "value": jc5["value"], "unit": UNIT,
                                        "ms_per_step": jc5["ms_per_step"], "l2": rc5["l2"], "filtered_blocks_per_s": None,
                                        "roofline": roofline_block(wi, rc5, jc5["ms_per_step"], peaks, hbm_peak),
                                        "clocks": rc5["clocks"], "gpu_launches": int(rc5["launches"])}
            torch.cuda.empty_cache()
        if world == 1 and not args.no_adaptive:
            others["adaptive_p6"] = time_adaptive(fe, torch, local, peaks, hbm_peak, min(args.steps, 5), 3)
            others["adaptive_p6_generic"] = time_adaptive(fe, torch, local, peaks, hbm_peak, min(args.steps, 5), 3, generic=True)
            torch.cuda.empty_cache()
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    line = {"metric": METRIC, "value": job["value"], "unit": UNIT, "n_gpus": job["n_gpus"], "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": job["ms_per_step"], "higher_is_better": True, "scaling": args.scaling,
            "vs_baseline": None, "dtype": "f64", "data": "stub" if args.stub else "synthetic",
            "config": {"workload": w.describe(), "columns_per_gpu": B, "columns_total": job["columns_total"],
                       "l2": r.get("l2"), "parallelism": "columns split over %d GPU(s), no collective" % world},
            "gpu_launches": int(r["launches"]),
            "e2e": {"value": job["e2e_value"], "unit": UNIT, "h2d_bytes_per_step": r["e2e_bytes"],
                    "d2h_bytes_per_step": r["e2e_bytes"], "steps": args.steps,
                    "how": "cheb_filter_host on a pinned HOST block: H2D, filter, D2H inside the timed region, every step"},
            "filtered_blocks_per_s": world / (job["ms_per_step"] * 1e-3) if w.m > 0 else None}
    if not args.stub:
        line["roofline"] = roofline_block(w, r, job["ms_per_step"], peaks, hbm_peak)
        line["clocks"] = r["clocks"]
        line["workloads"] = others
        line["peaks"] = peaks
        if args.orders and world == 1:
            line["orders"] = time_orders(fe, torch, local, peaks, hbm_peak, 3, 3)
            # the adaptive hanging-node mesh at the orders of the paper's Table 1: box-cell kernel and generic kernel
            line["orders_adaptive"] = {}
            for p_ in (4, 5, 6, 7):
                for generic in (False, True):
                    r_ = time_adaptive(fe, torch, local, peaks, hbm_peak, 3, 3, p=p_, m=12, generic=generic)
                    line["orders_adaptive"]["p%d%s" % (p_, "_generic" if generic else "")] = {
                        "value": r_["value"], "unit": UNIT, "ms_per_apply": r_["ms_per_step"] / 12, "frac": r_["roofline"]["frac"]}
                    torch.cuda.empty_cache()
        if args.consumers and world == 1:
            line["consumers"] = time_consumers(fe, torch, workloads.config(2), local)
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(args.workload, SAMPLE_CELLS[args.workload])
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
