#!/usr/bin/env python
"""bench.py -- WPCD hot path throughput on B200 (channel-solves/s), roofline of the dominant kernel, CPU-oracle baseline.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--samples S] [--N n_wp]

A "step" is one pass of the whole hot path (assembly -> batched diagonalisation -> on-shell T -> phase shifts) over
one batch of synthetic input: BASELINE.json config 5 at N=100, i.e. 4096 seeded samples of the perturbed two-Yukawa
potential x {1S0 (100x100), 3S1-3D1 (200x200)}, 350 energies.  The path does not shard (north_star: one GPU, no
collectives): --gpus N > 1 runs N independent replicas (weak scaling, no data-path collective).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2106_00454_b200 import inputs as inp  # noqa: E402

FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # 148 SMs x 64 FP64 FMA lanes x 2 flop x 1.965 GHz
# DRAM traffic per Jacobi launch comes from the committed ncu capture, keyed by (n, batch): profiles/jacobi_dram_traffic.csv
# (command in profiles/jacobi_dram_traffic.md).  It is a static figure of that capture, reported only when (n, batch) match.
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "jacobi_dram_traffic.csv")


def ncu_traffic(n, batch):
    """(bytes per launch or None, source/reason) from the committed profile table."""
    try:
        rows = [ln.strip().split(",") for ln in open(TRAFFIC_CSV) if ln.strip() and not ln.startswith("#")]
    except OSError:
        return None, "profiles/jacobi_dram_traffic.csv missing"
    for r in rows[1:]:
        if int(r[0]) == n and int(r[1]) == batch:
            return float(r[2]), f"dram__bytes_read.sum + dram__bytes_write.sum of one launch, {r[3]} (static: from the committed capture, not this run)"
    return None, f"no committed ncu capture for n={n}, batch={batch}"


def measure_fp64_peak(h, torch):
    """FP64 peak measured in this run with the library's register-only chain kernels (wpcd_probe_fp64): best of 3 launches
    each of DFMA chains and DMMA (mma.sync.m8n8k4.f64) chains, CUDA events on the launching stream."""
    out = {}
    for kind, name in ((0, "dfma"), (1, "dmma")):
        iters = 20000 if kind == 0 else 4000
        best, sink = 0.0, None
        for _ in range(4):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            flops, sink = h.probe_fp64(kind, iters, sink=sink)
            e1.record()
            torch.cuda.synchronize()
            best = max(best, flops / (e0.elapsed_time(e1) * 1e-3) / 1e12)
        out[name] = best
    return out


METRIC = "channel-solves/s (fp64 H diag + on-shell T at all E)"
CHANNELS = [(0, 0), (1, 1)]   # single 1S0 (n=N) and coupled 3S1-3D1 (n=2N)


def workload_name(N, S, nE):
    return f"config5@N={N}: {S} samples x {{1S0 {N}x{N}, 3S1-3D1 {2 * N}x{2 * N}}}, {nE} energies"


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""

    def __init__(self, gpu_index=0):
        super().__init__(daemon=True)
        self.gpu = gpu_index
        self.stop_flag = threading.Event()
        self.rows = []

    def run(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        while not self.stop_flag.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self.stop_flag.wait(0.2)

    def summary(self):
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        reasons = set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------- oracle (CPU) arm
def oracle_sample(N, nE, n_each, cores):
    """The CPU oracle, as it stands, on n_each (sample, 1S0) + n_each (sample, 3S1-3D1) solves of the same workload:
    assembly -> cyclic Jacobi -> on-shell T -> phases, one solve per thread.  Returns (solves, seconds)."""
    from concurrent.futures import ThreadPoolExecutor
    from oracle import oracle as o
    p = inp.grid_edges(N)
    e0, dE, Ee = o.fwp(p)
    tl, Ecm = inp.energies(nE)
    scales = inp.sample_scales(4096, seed=0)

    def one(job):
        s, coupled = job
        V0 = inp.MT_V0 * scales[s, :2]
        if not coupled:
            H, V = o.assemble_H(e0, o.V_yukawa(p, 0, V0, inp.MT_MU))
        else:
            H, V = o.assemble_H(e0, o.V_yukawa(p, 0, V0, inp.MT_MU), o.V_yukawa(p, 2, V0, inp.MT_MU),
                                o.V_yukawa(p, 1, [inp.TENSOR_V * scales[s, 2]], [inp.TENSOR_MU]))
        W, C, sw = o.jacobi(H)
        T, b = o.onshell_T(N, bool(coupled), Ee, V, W, C, Ecm)
        d, S = o.phase_shifts(bool(coupled), T, b, dE)
        return float(d.ravel()[0])

    jobs = [(s, 1) for s in range(n_each)] + [(s, 0) for s in range(n_each)]
    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=cores) as ex:
        list(ex.map(one, jobs))
    return len(jobs), time.perf_counter() - t0


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = os.cpu_count() or 1
    n_each = 16 * max(cores, 8)
    for _ in range(args.warmup):
        oracle_sample(args.N, args.nE, max(cores // 4, 1), cores)
    t0 = time.perf_counter()
    solves = 0
    for _ in range(args.steps):
        k, _dt = oracle_sample(args.N, args.nE, n_each, cores)
        solves += k
    dt = time.perf_counter() - t0
    val = solves / dt
    sample = f"{n_each} samples x (1S0 + 3S1-3D1) per step, threads over solves; same inputs as the GPU arm"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "channel-solves/s", "n_gpus": args.gpus,
            "ranks_working": 1,   # the oracle runs on rank 0's host cores only, whatever N the driver launched
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.N, args.samples, args.nE), "bounded_sample": sample},
            "cpu_baseline": {"value": val, "unit": "channel-solves/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "channel-solves/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------- GPU arm
def rows_fraction(pipe, kind):
    """Fraction of the rows of C that the pass needs (the rows wpcd_onshell_T reads): the algorithmic share of the
    eigenvector update.  The kernel updates whole 8-row blocks of its internal ordering, i.e. slightly more."""
    rows, n = pipe.rows[kind], pipe.kind[kind]["n"]
    if rows is None:
        return 1.0
    return sum(hi - lo for lo, hi in rows) / float(n)


def jacobi_flops(n, f):
    """Algorithmic flops of one Jacobi sweep: n(n-1)/2 rotations x (6n for the symmetric A + 6n f for C) ~ (3 + 3f) n^3."""
    return (3.0 + 3.0 * f) * n ** 3


def max_over_ranks(values, world, device):
    """Replicas only: the one cross-rank step of the bench is the MAX of the per-rank timings."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2106_00454_b200.pipeline import Pipeline

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the WPCD path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    N, S, nE = args.N, args.samples, args.nE
    if args.workload == "config3":          # BASELINE.json config 3: the Bayesian-sampling batch, all 14 channels J <= 4
        N, S = 100, (1024 if args.samples == 4096 else args.samples)
        channels = [(c, l) for _, c, l in inp.CHANNELS_J4]
        wname = f"config3: {S} samples x 14 channels J<=4 (10 of {N}x{N}, 4 of {2 * N}x{2 * N}), {nE} energies"
    else:
        channels = CHANNELS
        wname = workload_name(N, S, nE)
    tl, Ecm = inp.energies(nE)
    # every replica gets its own seeded batch (replicas only: the path does not shard)
    scales = inp.sample_scales(S, seed=rank)
    pot = dict(V0=inp.MT_V0, mu=inp.MT_MU, scale_idx=[0, 1], VT=inp.TENSOR_V, muT=inp.TENSOR_MU, VT_scale_idx=2)
    pipe = Pipeline(inp.grid_edges(N), channels, Ecm, S, pot, device=local)
    pipe.scales.copy_(torch.as_tensor(scales))
    names = pipe.stage_names()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        pipe.solve_device()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    ev = [{nm: (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for nm in names}
          for _ in range(args.steps)]
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0.record()
    for k in range(args.steps):
        pipe.solve_device(events=ev[k])
    t1.record()
    barrier()
    ms = t0.elapsed_time(t1)
    stage_ms = {nm: float(np.mean([e[nm][0].elapsed_time(e[nm][1]) for e in ev])) for nm in names}
    info = {k: b["info"].cpu().numpy() for k, b in pipe.kind.items()}
    if any((v < 1).any() for v in info.values()):
        raise SystemExit("bench.py: Jacobi did not converge on some matrix")

    # end to end through the public API with host buffers (pinned), copies inside the timed region
    for _ in range(2):
        pipe.solve_host(scales)
    barrier()
    te0 = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        pipe.solve_host(scales)
    e1.record()
    barrier()
    ms_e2e = max(e0.elapsed_time(e1), 1e3 * (time.perf_counter() - te0))
    if sampler:
        sampler.stop_flag.set()
        sampler.join()

    ms, ms_e2e = max_over_ranks([ms, ms_e2e], world, "cuda")
    solves = pipe.channel_solves * world
    value = solves * args.steps / (ms * 1e-3)
    e2e = solves * args.steps / (ms_e2e * 1e-3)

    if rank == 0:
        # dominant kernel = the Jacobi launch with the larger share; algorithmic flops = 6 n^3 x rotating sweeps
        dom = max((nm for nm in names if nm.startswith("diag_")), key=lambda nm: stage_ms[nm])
        kind = 1 if dom.endswith("cpl") else 0
        n = pipe.kind[kind]["n"]
        rot_sweeps = float(np.mean(info[kind] - 1))          # the last sweep only verifies convergence
        flops = jacobi_flops(n, rows_fraction(pipe, kind)) * rot_sweeps * pipe.kind[kind]["batch"]
        ach = flops / (stage_ms[dom] * 1e-3) / 1e12
        jac = {}
        for k2, b in pipe.kind.items():
            nm = "diag_cpl" if k2 else "diag_unc"
            f = jacobi_flops(b["n"], rows_fraction(pipe, k2)) * float(np.mean(info[k2] - 1)) * b["batch"]
            jac[nm] = {"n": b["n"], "batch": b["batch"], "ms": stage_ms[nm], "rotating_sweeps": float(np.mean(info[k2] - 1)),
                       "rows_of_C_needed": rows_fraction(pipe, k2),
                       "tflops_algorithmic": f / (stage_ms[nm] * 1e-3) / 1e12,
                       "frac_fp64_peak": f / (stage_ms[nm] * 1e-3) / 1e12 / FP64_PEAK_TFLOPS}
        peak_meas = measure_fp64_peak(pipe.h, torch)
        traffic, traffic_src = ncu_traffic(n, pipe.kind[kind]["batch"])
        # secondary (HBM) rooflines: assembly stage and on-shell stage, algorithmic bytes over the stage's event time
        hbm_peak = None
        try:
            hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
        except Exception:
            pass
        hbm_src = "MEASURED_PEAKS.json hbm_gbs" if hbm_peak else "fallback 6551.7 GB/s (this pool's measured copy bandwidth, B200_PROFILING.md)"
        hbm_peak = hbm_peak or 6551.7
        secondary = []
        bytes_H = sum(8.0 * b["n"] ** 2 * b["batch"] for b in pipe.kind.values())
        secondary.append({"bound": "hbm", "kernel": "assembly stage (k_grid + k_basis + k_combine): write H", "achieved": bytes_H / (stage_ms["build"] * 1e-3) / 1e9,
                          "peak": hbm_peak, "unit": "GB/s", "frac": bytes_H / (stage_ms["build"] * 1e-3) / 1e9 / hbm_peak,
                          "bytes_model": "8 n^2 per channel-solve (H written once)", "peak_source": hbm_src})
        for k2, b in pipe.kind.items():
            nm = "onshell_cpl" if k2 else "onshell_unc"
            f2 = rows_fraction(pipe, k2) if b["n"] <= 200 else 1.0
            by = (8.0 * b["n"] ** 2 * f2 + 8.0 * b["n"] + 16.0 * nE * (4 if k2 else 1) + 8.0 * nE * (3 if k2 else 1)) * b["batch"]
            if b["n"] > 200:
                by += 8.0 * b["n"] ** 2 * rows_fraction(pipe, k2) * b["batch"]       # the on-shell rows of H for V C
            secondary.append({"bound": "hbm", "kernel": f"on-shell stage ({nm}: k_onshell + k_phase, n={b['n']})",
                              "achieved": by / (stage_ms[nm] * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                              "frac": by / (stage_ms[nm] * 1e-3) / 1e9 / hbm_peak,
                              "bytes_model": "rows of C the contraction reads + W + T and delta out", "peak_source": hbm_src})
        cpu = None
        if world == 1 and not args.no_cpu_baseline and args.workload == "bench":
            cores = os.cpu_count() or 1
            n_each = 64 * max(cores, 8)          # about 10-20 s of CPU work on the box's cores
            k, dt = oracle_sample(N, nE, n_each, cores)
            cpu = {"value": k / dt, "unit": "channel-solves/s", "cores": cores, "kind": "oracle",
                   "sample": f"{n_each} samples x (1S0 + 3S1-3D1) of the same workload, one solve per thread, {dt:.1f} s"}
        line = {"metric": METRIC, "value": value, "unit": "channel-solves/s", "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": wname, "l2": "inputs_exceed_L2 (H batch >> 126 MB)",
                           "replicas": world, "jacobi_tol": "2^-52 relative pivot test", "n_gl": 8},
                "clocks": sampler.summary() if sampler else None,
                "e2e": {"value": e2e, "unit": "channel-solves/s", "h2d_bytes_per_step": pipe.h2d_bytes(),
                        "d2h_bytes_per_step": pipe.d2h_bytes(), "ms_per_step": ms_e2e / args.steps},
                "gpu_launches": pipe.launches_per_step * args.steps,
                "roofline": {"bound": "alu", "kernel": f"k_jacobi ({dom}, n={n})", "achieved": ach, "peak": FP64_PEAK_TFLOPS,
                             "unit": "TFLOP/s", "frac": ach / FP64_PEAK_TFLOPS, "traffic": traffic, "traffic_source": traffic_src,
                             "algorithmic_bytes": (16.0 * n * n + 8.0 * n) * pipe.kind[kind]["batch"],
                             "peak_source": "derived: 148 SM x 64 FP64 FMA/clk x 2 x 1.965 GHz (DESIGN.md section 6); MEASURED_PEAKS.json has no fp64 entry",
                             "peak_measured": peak_meas, "peak_measured_source": "wpcd_probe_fp64 in this run: register-only DFMA / DMMA chains on all SMs, best of 4, CUDA events",
                             "frac_of_measured": ach / max(peak_meas.values()),
                             "flops_model": "(3 + 3 f) n^3 x rotating sweeps x batch: 3 n^3 for A (symmetric), 3 n^3 for the eigenvectors "
                                            "(SURVEY 8(d): 6 n^3), the latter scaled by the fraction f of rows of C that the on-shell step needs"},
                "roofline_secondary": secondary, "stages_ms": stage_ms, "jacobi": jac, "cpu_baseline": cpu}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_table1(args):
    """Context only (not the bench metric): the regime of the paper's Table 1 -- all 14 channels J <= 4,
    Chebyshev momentum bins (Eq. 31), mid-point potential (Eq. 30), energy-averaged T (Eq. 28) at 350 energies, phase
    shifts and total cross section -- as wall time per potential sample for N_WP = 16, 24, 32, 96; one sample (latency)
    and 1024 samples (throughput).  The paper: 0.5 / 2.5 / 6 / 35 ms on a V100 for one sample with a pre-computed V."""
    import torch
    from paper_2106_00454_b200.pipeline import Pipeline
    names = [c[0] for c in inp.CHANNELS_J4]
    channels = [(c[1], c[2]) for c in inp.CHANNELS_J4]
    _, Ecm = inp.energies(350)
    pot = dict(V0=inp.MT_V0, mu=inp.MT_MU, scale_idx=[0, 1], VT=inp.TENSOR_V, muT=inp.TENSOR_MU, VT_scale_idx=2)
    out = {}
    # "exact" reference: the MI method on the same GPU (wpcd_mi_solve, N_Q = 48), sample 0 (scales of seed 0)
    from paper_2106_00454_b200 import wpcd
    h = wpcd.Handle(0)
    dE = torch.as_tensor(np.ascontiguousarray(Ecm), device="cuda:0")
    sc0 = torch.as_tensor(inp.sample_scales(1, seed=0), device="cuda:0")
    J = [inp.channel_sJ(nm)[1] for nm in names]
    Ju = [j for (c, _), j in zip(channels, J) if not c]; Jc = [j for (c, _), j in zip(channels, J) if c]
    torch.cuda.synchronize(); t0 = time.perf_counter()
    S_unc, S_cpl = h.mi_solve(channels, dE, NQ=48, scales=sc0, S=1, **pot)
    sig_mi = h.sigma_tot(Ju, S_unc, Jc, S_cpl, None, None, dE)[0]
    torch.cuda.synchronize(); mi_ms = 1e3 * (time.perf_counter() - t0)
    tlab = 2.0 * Ecm
    sel = torch.as_tensor(tlab >= 40.0, device="cuda:0")
    cE = inp.HBARC ** 2 / (2 * inp.MU)
    qt = torch.as_tensor(np.sqrt(Ecm / cE), device="cuda:0")            # target momenta
    for N in (16, 24, 32, 96):
        edges = inp.grid_chebyshev(N)
        qmid = 0.5 * (edges[:-1] + edges[1:])
        for S in (1, 1024):
            # the production variant: ONE energy-averaged T per bin, evaluated at the bin mid-points
            # q_i, then linear interpolation between the mid-points (here of sigma_tot, with torch ops: context only)
            pipe = Pipeline(edges, channels, cE * qmid ** 2, S, pot, device=0, mode=1, n_gl=1,
                            channel_J=[inp.channel_sJ(nm)[1] for nm in names])
            pipe.scales.copy_(torch.as_tensor(inp.sample_scales(S, seed=0)))
            for _ in range(3):
                pipe.solve_device()
            torch.cuda.synchronize()
            reps = 20 if S == 1 else 5
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(reps):
                pipe.solve_device()
            e1.record(); torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / reps
            assert all(int((b["info"] < 1).sum()) == 0 for b in pipe.kind.values())
            ms_graph = None
            if S == 1:      # one sample is launch/latency bound: the same pass replayed as a CUDA graph
                sig_ref = pipe.sigma.clone()
                replay = pipe.capture()
                for _ in range(3):
                    replay()
                torch.cuda.synchronize()
                e0.record()
                for _ in range(reps):
                    replay()
                e1.record(); torch.cuda.synchronize()
                ms_graph = e0.elapsed_time(e1) / reps
                assert torch.equal(torch.nan_to_num(pipe.sigma), torch.nan_to_num(sig_ref))
            qm = torch.as_tensor(qmid, device="cuda:0")
            i1 = torch.clamp(torch.searchsorted(qm, qt), 1, N - 1); i0 = i1 - 1
            w = (qt - qm[i0]) / (qm[i1] - qm[i0])
            sig = pipe.sigma[0, i0] * (1 - w) + pipe.sigma[0, i1] * w          # sample 0 has the scales of the MI reference
            d = sig - sig_mi
            rmse = float(torch.sqrt((d ** 2).mean()))                            # Eq. 44, 1..350 MeV
            rmse40 = float(torch.sqrt((d[sel] ** 2).mean()))                     # 40..350 MeV
            out[f"N_WP={N},S={S}"] = {"ms_per_pass": ms, "ms_per_pass_cuda_graph": ms_graph, "ms_per_sample": ms / S, "rmse_sigma_tot_mb": rmse,
                                      "rmse_sigma_tot_mb_40_350MeV": rmse40}
    print(json.dumps({"workload": "paper_table1 (context, not the bench metric)", "channels": 14, "energies": 350,
                      "variant": "Chebyshev bins, mid-point V, energy-averaged T at the bin mid-points, phases, sigma_tot, linear interpolation to 350 energies; RMSE (Eq. 44) against MI on the GPU",
                      "mi_reference": {"N_Q": 48, "ms_one_sample_incl_sigma": mi_ms}, "results": out,
                      "paper": {"hardware": "Tesla V100, one sample, pre-computed V", "ms": {"16": 0.5, "24": 2.5, "32": 6, "96": 35}}}))


def run_config5_sweep(args):
    """BASELINE.json config 5 in full: N in {32 ... 400} x 4096 seeded samples x {1S0 N x N, 3S1-3D1 2N x 2N}, 350 energies,
    on the GPU (channel-solves/s, Jacobi fraction of the FP64 peak per launch), "plus the MI solver on the CPU oracle at
    the same N for method-error and wall-time comparison" (SURVEY 8(d) "Oracle timing": N_Q = N, one sample, the same
    energies; Eq. 37, 435-449 Table 1).  Prints ONE JSON object with all N."""
    import torch
    from concurrent.futures import ThreadPoolExecutor
    from paper_2106_00454_b200.pipeline import Pipeline
    from oracle import oracle as o
    cores = os.cpu_count() or 1
    nE, S = args.nE, args.samples
    tl, Ecm = inp.energies(nE)
    scales = inp.sample_scales(S, seed=0)
    pot = dict(V0=inp.MT_V0, mu=inp.MT_MU, scale_idx=[0, 1], VT=inp.TENSOR_V, muT=inp.TENSOR_MU, VT_scale_idx=2)
    d180 = lambda a, b: np.abs((a - b + 90.0) % 180.0 - 90.0)
    rows = {}
    peak = None
    for N in [int(x) for x in args.sweep_N.split(",")]:
        pipe = Pipeline(inp.grid_edges(N), CHANNELS, Ecm, S, pot, device=0)
        if peak is None:
            peak = measure_fp64_peak(pipe.h, torch)
        pipe.scales.copy_(torch.as_tensor(scales))
        names = pipe.stage_names()
        for _ in range(max(args.warmup, 3) if N <= 200 else 1):
            pipe.solve_device()
        torch.cuda.synchronize()
        steps = args.steps if N <= 200 else max(1, min(args.steps, 2))
        ev = [{nm: (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for nm in names} for _ in range(steps)]
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record()
        for k in range(steps):
            pipe.solve_device(events=ev[k])
        t1.record()
        torch.cuda.synchronize()
        ms = t0.elapsed_time(t1) / steps
        stage_ms = {nm: float(np.mean([e[nm][0].elapsed_time(e[nm][1]) for e in ev])) for nm in names}
        info = {k: b["info"].cpu().numpy() for k, b in pipe.kind.items()}
        assert all((v >= 1).all() for v in info.values()), "Jacobi did not converge"
        jac = {}
        for k2, b in pipe.kind.items():
            nm = "diag_cpl" if k2 else "diag_unc"
            f = jacobi_flops(b["n"], rows_fraction(pipe, k2)) * float(np.mean(info[k2] - 1)) * b["batch"]
            jac[nm] = {"n": b["n"], "ms": stage_ms[nm], "rotating_sweeps": float(np.mean(info[k2] - 1)),
                       "frac_fp64_peak": f / (stage_ms[nm] * 1e-3) / 1e12 / FP64_PEAK_TFLOPS}
        d_unc = pipe.kind[0]["delta"][0].cpu().numpy()            # sample 0 (scales of seed 0, row 0)
        d_cpl = pipe.kind[1]["delta"][0].cpu().numpy()
        del pipe
        torch.cuda.empty_cache()
        # ---- MI on the CPU oracle: N_Q = N, sample 0, the same energies (a stride subsample above N = 200, stated)
        n_mi = args.mi_energies or nE
        idx = np.unique(np.linspace(0, nE - 1, n_mi).round().astype(int))
        V0 = inp.MT_V0 * scales[0, :2]

        def mi_one(e):
            Su, _ = o.mi_solve(tl[e], V0=V0, mu=inp.MT_MU, l_or_J=0, NQ=N)
            Sc, _ = o.mi_solve(tl[e], coupled=True, V0=V0, mu=inp.MT_MU, l_or_J=1, VT=inp.TENSOR_V * scales[0, 2], muT=inp.TENSOR_MU, NQ=N)
            return Su, Sc
        w0 = time.perf_counter()
        with ThreadPoolExecutor(max_workers=cores) as ex:
            res = list(ex.map(mi_one, idx))
        mi_s = time.perf_counter() - w0
        # ---- the same MI systems on the GPU (wpcd_mi_solve: K-matrix form), where one CTA can take them
        mi_gpu = None
        try:
            from paper_2106_00454_b200 import wpcd as _w
            hg = _w.Handle(0)
            dEc = torch.as_tensor(np.ascontiguousarray(Ecm), device="cuda:0")
            sc0 = torch.as_tensor(scales[:1].copy(), device="cuda:0")
            # one thread per row: both channels up to N_Q = 127 (above 81 with the system in an L2 region), 1S0 alone up to 255
            chans = [(0, 0), (1, 1)] if N <= 127 else [(0, 0)] if N <= 255 else []
            if chans:
                for _ in range(2):
                    hg.mi_solve(chans, dEc, NQ=N, scales=sc0, S=1, **pot)
                torch.cuda.synchronize()
                g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                g0.record(); Sg_u, Sg_c = hg.mi_solve(chans, dEc, NQ=N, scales=sc0, S=1, **pot); g1.record(); torch.cuda.synchronize()
                Su = Sg_u.cpu().numpy()[0, 0]; Su = Su[..., 0] + 1j * Su[..., 1]
                mi_gpu = {"channels": "1S0 + 3S1-3D1" if len(chans) == 2 else "1S0 only (coupled system: more rows than threads of a CTA)",
                          "ms_per_sample_350_energies": g0.elapsed_time(g1),
                          "max_abs_dS_vs_cpu_oracle_1S0": float(np.abs(Su[idx] - np.array([r[0] for r in res])).max())}
            hg.close()
        except Exception as ex:  # context leg only: never fails the sweep
            mi_gpu = {"error": str(ex)[:200]}
        du = np.array([0.5 * np.degrees(np.angle(r[0])) for r in res])
        dc = np.array([[0.5 * np.degrees(np.angle(r[1][0, 0])), 0.5 * np.degrees(np.angle(r[1][1, 1]))] for r in res])
        eu = d180(d_unc[idx], du)
        ec = d180(d_cpl[idx][:, :2], dc)
        rows[str(N)] = {"ms_per_step": ms, "channel_solves_per_s": 2 * S / (ms * 1e-3), "stages_ms": stage_ms, "jacobi": jac,
                        "mi_cpu_oracle": {"N_Q": N, "energies_solved": int(len(idx)), "wall_s": mi_s,
                                          "wall_s_per_sample_350_energies": mi_s * nE / len(idx), "cores": cores,
                                          "systems": "1S0 (N_Q+1 complex) + 3S1-3D1 (2 N_Q + 2 complex) per energy"},
                        "mi_gpu": mi_gpu,
                        "wpcd_gpu_ms_per_sample_in_batch": ms / S,
                        "method_error_deg": {"1S0_median": float(np.median(eu)), "1S0_max": float(eu.max()),
                                             "3S1_3D1_delta_median": float(np.median(ec)), "3S1_3D1_delta_max": float(ec.max())}}
    print(json.dumps({"workload": "config5_sweep: N x 4096 samples x {1S0, 3S1-3D1}, 350 energies; MI on the CPU oracle at N_Q = N",
                      "metric": METRIC, "unit": "channel-solves/s", "samples": S, "energies": nE, "dtype": "f64",
                      "fp64_peak": {"derived_tflops": FP64_PEAK_TFLOPS, "measured_tflops": peak}, "results": rows}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--samples", type=int, default=4096)
    ap.add_argument("--N", type=int, default=100)
    ap.add_argument("--nE", type=int, default=350)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--workload", default="bench", choices=["bench", "config3", "config5_sweep", "paper_table1"])
    ap.add_argument("--sweep-N", default="32,48,64,100,150,200,300,400", help="config5_sweep: the N values")
    ap.add_argument("--mi-energies", type=int, default=0, help="config5_sweep: energies the CPU MI leg solves per N (0 = all)")
    args = ap.parse_args()
    if args.workload == "paper_table1":
        return run_table1(args)
    if args.workload == "config5_sweep":
        return run_config5_sweep(args)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
