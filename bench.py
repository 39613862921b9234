#!/usr/bin/env python
"""bench.py -- throughput of the fused Chebyshev-filter H~X path on the BASELINE.json workloads.

A "step" is one cheb_filter call (m fused operator steps: gather -> cell contraction -> scatter + recurrence) on
one block of B vectors.  metric = GDoF-vectors/s = N_free * B * m * steps / time (reading R14).  Prints ONE JSON
line (rank 0).  See DESIGN.md "Measurement" for the roofline arithmetic.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 2|3|4|5] [--extra] [--impl reference]
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
# FP64 ALU roofline: 148 SMs x 64 DFMA/clk/SM x 2 flop x 1.965 GHz (MEASURED_PEAKS.json sm_max_mhz)
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


# dram__bytes_read.sum + dram__bytes_write.sum of ONE k_apply_tma launch from the committed `ncu --set full` captures
# (profiles/r1b_c2_k_apply_tma_full.md, profiles/r1b_c3_k_apply_tma_full.md)
NCU_TRAFFIC_BYTES = {2: 296.28e6 + 221.12e6, 3: 3.4418e9 + 3.1540e9}


def algorithmic_flops_per_cell_vector(p):
    """matrix-free sum factorisation, 24 n^4 + 9 n^3 flops per cell-vector."""
    n = p + 1
    return 24 * n**4 + 9 * n**3


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
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            parts = [s.strip() for s in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for nme, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nme)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm))
        return out


def cpu_baseline(w_index, budget_cells, steps=1, all_cores=True):
    """The oracle as it stands, on a bounded sample: the same recipe on a centred sub-mesh of budget_cells^3 cells,
    all B columns, full degree m (config 5: 4 shifted applies).  Setup (cell matrices, CSR) is not timed."""
    import oracle
    w = workloads.reduced(w_index, budget_cells)
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
           "sample": "%s: centred %d^3-cell sub-mesh (N=%d), all B=%d columns, %d applies, serial CSR oracle; setup untimed"
                     % (w.name, budget_cells, om.N, w.B, napply),
           "seconds_per_step": t1}
    if all_cores:
        nc = os.cpu_count() or 1
        tn = run(nc)
        out["value_all_cores"] = om.N_free * w.B * napply / tn / 1e9
        out["cores_all"] = nc
    return out


SAMPLE_CELLS = {2: 6, 3: 4, 4: 4, 5: 6}


def run_reference(args):
    """--impl reference: the oracle timed on the host cores, same metric / config; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = workloads.config(args.workload)
    for _ in range(min(args.warmup, 1)):
        cpu_baseline(args.workload, 2, 1, all_cores=False)
    cb = cpu_baseline(args.workload, SAMPLE_CELLS[args.workload], max(1, args.steps), all_cores=False)
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": cb["seconds_per_step"] * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.describe(), "sample": cb["sample"]},
            "cpu_baseline": {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def time_workload(fe, torch, w, steps, warmup, dev, seed_offset=0, with_e2e=False, dist=None, sample_clocks=False,
                  variant=0):
    """Device-resident timing of `steps` cheb_filter calls (config 5: blocks of 200 shifted applies)."""
    gm = fe.FEMesh(w.xe, w.ye, w.ze, w.p, device=dev)
    if variant:
        gm.set_variant(variant)
    Vq = w.V(gm.quad_coords())
    gm.set_potential(Vq)
    mask = torch.as_tensor(gm.mask().astype(np.float64), device="cuda")[:, None]
    N, B = gm.N, w.B
    nrot = 3 if N * B * 8 < 1 << 30 else 1  # rotate buffer sets when one block is L2-scale (config 2/5)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(1234 + w.x_seed + seed_offset)
    pristine = torch.randn(N, B, dtype=torch.float64, device="cuda", generator=gen) * mask
    Xs = [torch.empty_like(pristine) for _ in range(nrot)]
    works = [torch.empty(2 * N * B, dtype=torch.float64, device="cuda") for _ in range(nrot)]
    a0, a, b = spectrum_bounds(w)
    eps = torch.as_tensor(w.eps(), device="cuda") if w.eps_seed is not None else None
    napply = w.m if w.m > 0 else w.n_applies

    def one_step(i):
        X, wk = Xs[i % nrot], works[i % nrot]
        if w.m > 0:
            gm.cheb_filter(X, w.m, a, b, a0, wk)
        else:  # R19: alternate two input and two output blocks
            Y0, Y1 = wk[:N * B].view(N, B), wk[N * B:].view(N, B)
            for t in range(w.n_applies):
                gm.apply_H(X if t % 2 == 0 else pristine, Y0 if t % 2 == 0 else Y1, eps)

    def restore(i):  # only the block the coming step filters
        Xs[i % nrot].copy_(pristine)

    for i in range(warmup):
        restore(i)
        one_step(i)
    torch.cuda.synchronize()
    sampler = ClockSampler(dev) if sample_clocks else None
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
    clocks = sampler.stop() if sampler else None
    ms = [e0.elapsed_time(e1) for e0, e1 in ev]
    total_ms = float(sum(ms))
    res = {"gm": gm, "ms_per_step": total_ms / steps, "ms_min": float(min(ms)), "launches": gm.launches - l0,
           "napply": napply, "N": N, "N_free": gm.N_free, "B": B, "clocks": clocks, "ncells": gm.ncells}
    if with_e2e:
        # end to end through the public API with HOST buffers: pinned H2D of the block, filter, D2H of the result
        host_in = pristine.cpu().pin_memory()
        host_out = torch.empty_like(host_in).pin_memory()
        X, wk = Xs[0], works[0]
        e2e_steps = max(1, min(steps, 3))

        def e2e_step():
            if w.m > 0:  # the C-ABI host-buffer call: H2D, filter, D2H (column chunks pipelined), synchronous
                gm.cheb_filter_host(host_io, w.m, a, b, a0)
            else:
                X.copy_(host_in, non_blocking=True)
                one_step(0)
                host_out.copy_(wk[:N * B].view(N, B), non_blocking=True)

        host_io = host_in.clone().pin_memory() if w.m > 0 else None
        e2e_step()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            e2e_step()
        torch.cuda.synchronize()
        res["e2e_s_per_step"] = (time.perf_counter() - t0) / e2e_steps
        res["e2e_bytes"] = host_in.numel() * 8
    return res


def time_consumers(fe, torch, w, dev):
    """NEXT-1 / NEXT-2 on the workload's mesh (informational, --extra): one Rayleigh-Ritz call on a filtered block and
    a fixed number of preconditioned MINRES steps with the config-5 shifts."""
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
    return {"mesh": w.describe(), "rayleigh_ritz_ms": rr_ms, "gram_ms": gram_ms,
            "gram_tflops": 2.0 * N * B * B / (gram_ms * 1e-3) / 1e12, "gram_gbs": 16.0 * N * B / (gram_ms * 1e-3) / 1e9,
            "minres_ms_per_step": mr_ms, "minres_steps_timed": it}


def summarize(w, r, total_ms_per_step, n_ranks=1):
    dofvec = r["N_free"] * r["B"] * r["napply"] * n_ranks
    value = dofvec / (total_ms_per_step * 1e-3) / 1e9
    flops_launch = algorithmic_flops_per_cell_vector(w.p) * r["ncells"] * r["B"]
    dur = total_ms_per_step * 1e-3 / r["napply"]
    ach = flops_launch / dur / 1e12
    return value, {"bound": "alu", "achieved": ach, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                   "frac": ach / FP64_PEAK_TFLOPS, "traffic": None,
                   "kernel": "k_apply_tma<p=%d> (one fused operator step: filter time / m, CUDA events on the launching stream)" % w.p,
                   "launch_ms": dur * 1e3,
                   "peak_source": "derived: 148 SM x 64 DFMA/clk x 2 x 1.965 GHz (DESIGN.md); DFMA microbenchmark 36.8",
                   "hbm_frac_of_measured": None}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", type=int, default=2, choices=[2, 3, 4, 5])
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--extra", action="store_true", help="also time the other roofline workloads (3, 4, 5)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--variant", type=int, default=0)
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    import paper_2510_10529_b200 as fe
    fe.load_library()  # fails loudly if the CUDA extension is missing
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    w = workloads.config(args.workload)
    r = time_workload(fe, torch, w, args.steps, args.warmup, local, seed_offset=rank, with_e2e=True, dist=dist,
                      sample_clocks=(rank == 0), variant=args.variant)
    from paper_2510_10529_b200.colsplit import max_over_ranks
    # max over ranks; columns are sharded with no exchange (weak scaling)
    ms_step, e2e_ms = max_over_ranks([r["ms_per_step"], r["e2e_s_per_step"] * 1e3], dist, device="cuda")
    value, roof = summarize(w, r, ms_step, world)
    hbm_peak = None
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            hbm_peak = json.load(f)["hbm_gbs"]
    except Exception:
        pass
    alg_bytes = (24 if w.m > 0 else 16) * r["N"] * r["B"]
    roof["traffic"] = NCU_TRAFFIC_BYTES.get(args.workload)
    roof["algorithmic_bytes"] = alg_bytes
    roof["hbm_frac_of_measured"] = (alg_bytes / (roof["launch_ms"] * 1e-3) / 1e9 / hbm_peak) if hbm_peak else None
    ck = r.get("clocks") or {}
    if ck.get("sm_mhz") and ck.get("sm_max_mhz"):
        # the FP64 peak above assumes the maximum SM clock; long runs sit in sw_power_cap below it
        roof["frac_at_sampled_clock"] = roof["frac"] * ck["sm_max_mhz"] / ck["sm_mhz"]
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.describe(), "columns_per_gpu": w.B,
                       "l2": "3 rotating buffer sets, 3 x 141 MB blocks per filter > 126 MB L2" if r["N"] * r["B"] * 8 < 1 << 30
                       else "blocks of %.2f GB >> L2" % (r["N"] * r["B"] * 8 / 1e9),
                       "parallelism": "columns split over %d GPU(s), no collective" % world},
            "roofline": roof, "clocks": r["clocks"], "gpu_launches": int(r["launches"]),
            "e2e": {"value": r["N_free"] * r["B"] * r["napply"] * world / (e2e_ms * 1e-3) / 1e9, "unit": UNIT,
                    "h2d_bytes_per_step": r["e2e_bytes"], "d2h_bytes_per_step": r["e2e_bytes"]},
            "filtered_blocks_per_s": world / (ms_step * 1e-3) if w.m > 0 else None}
    del r["gm"]
    torch.cuda.empty_cache()
    if args.extra and world == 1:
        extra = {}
        for idx in (3, 4, 5):
            if idx == args.workload:
                continue
            wi = workloads.config(idx)
            try:
                ri = time_workload(fe, torch, wi, 2 if idx == 4 else 3, 1 if idx == 4 else 2, local, variant=args.variant)
                vi, rfi = summarize(wi, ri, ri["ms_per_step"])
                extra["cfg%d" % idx] = {"workload": wi.describe(), "value": vi, "unit": UNIT, "ms_per_step": ri["ms_per_step"],
                                        "roofline_frac": rfi["frac"], "achieved_tflops": rfi["achieved"]}
                del ri
            except Exception as ex:  # e.g. out of memory on a smaller part
                extra["cfg%d" % idx] = {"error": str(ex)[:200]}
            torch.cuda.empty_cache()
        line["other_workloads"] = extra
        try:
            line["consumers"] = time_consumers(fe, torch, w, local)
        except Exception as ex:
            line["consumers"] = {"error": str(ex)[:200]}
        torch.cuda.empty_cache()
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(args.workload, SAMPLE_CELLS[args.workload])
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
