#!/usr/bin/env python
"""bench.py -- throughput of the spectral Poisson hot path on B200 (BASELINE.json metric: grid
points/s per Poisson solve, 3-D unbounded fp32, and % of the HBM roofline).

One "step" = one pass of the whole hot path S1..S5 (X forward, Y forward, Z forward x Green's
spectrum x Z backward, Y backward, X backward) = one ``sf_solve`` through
the C ABI on one batch of synthetic input.  The workload is BASELINE.json configs[3]: 3-D unbounded
Poisson, 256^3 cell-centre grid zero-padded to 512^3 (Hockney-Eastwood), fp32, 16 seeded Gaussian
blobs, the Green's spectrum precomputed once at plan time and reused by every solve.
The paper times exactly this region (forward transform + convolution + backward transform, mean of
repeated runs).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl reference]

N > 1 (under torchrun): every rank solves its own independent problem (replicas only, DESIGN.md
"Multi-GPU"); no data-path collective; value = points of all ranks / max-over-ranks time.

``--impl reference`` times the CPU oracle (oracle/, plain fp64 C) on the host cores instead; it is
the only leg besides ``cpu_baseline`` that executes anything under oracle/.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "grid points/s per Poisson solve"
UNIT = "points/s"

# ---------------------------------------------------------------------------------------- workloads
# name -> (config number, n, precision, call); algorithmic bytes come from model_bytes() below
WORKLOADS = {
    "cfg1_periodic2d_64_f64_grad": dict(cfg=1, n=64, prec="f64", kind="periodic", call="gradient", ncomp=1, ndim=2),
    "cfg4_unbounded_256_f32": dict(cfg=4, n=256, prec="f32", kind="unbounded", call="solve", ncomp=1),
    "cfg4_unbounded_256_f64": dict(cfg=4, n=256, prec="f64", kind="unbounded", call="solve", ncomp=1),
    "cfg2_periodic_256_f32": dict(cfg=2, n=256, prec="f32", kind="periodic", call="solve", ncomp=1),
    "cfg2_periodic_256_f32_grad": dict(cfg=2, n=256, prec="f32", kind="periodic", call="gradient", ncomp=1),
    "cfg2_periodic_256_f64_grad": dict(cfg=2, n=256, prec="f64", kind="periodic", call="gradient", ncomp=1),
    "cfg3_dirichlet_255_f64": dict(cfg=3, n=255, prec="f64", kind="dirichlet", call="solve", ncomp=1),
    "cfg3_neumann_256_f64": dict(cfg=3, n=256, prec="f64", kind="neumann", call="solve", ncomp=1),
    "cfg5_vector_512_f32_curl": dict(cfg=5, n=512, prec="f32", kind="unbounded", call="curl", ncomp=3),
    "cfg5_vector_128_f32_curl": dict(cfg=5, n=128, prec="f32", kind="unbounded", call="curl", ncomp=3),
}
DEFAULT_WORKLOAD = "cfg4_unbounded_256_f32"


def model_bytes(w):
    """Algorithmic HBM bytes per step of each of the five kernels: every pass reads its input once and
    writes its output once, pruned (zero rows are neither read nor written), plus the compact Green's
    table in S3."""
    n, r = w["n"], (4 if w["prec"] == "f32" else 8)
    c = 2 * r
    nc = w["ncomp"]
    if w.get("ndim", 3) == 2:   # S1, the fused pass along y, S5 (periodic, gradient: three output fields)
        h = n // 2 + 1
        nout = 3 if w["call"] == "gradient" else 1
        spec = n * h * c
        return [n * n * r + spec, 0, spec + nout * spec, 0, nout * (spec + n * n * r)]
    if w["kind"] == "unbounded":
        hx, p = n + 1, 2 * n
        nout = nc
        s1 = nc * (n * n * n * r + n * n * hx * c)
        s2 = nc * (n * n * hx * c + n * p * hx * c)
        s3 = nc * (n * p * hx * c) + nout * (n * p * hx * c) + (n + 1) * (n + 1) * hx * r
        s4 = nout * (n * p * hx * c + n * n * hx * c)
        s5 = nout * (n * n * hx * c + n * n * n * r)
    elif w["kind"] == "periodic":
        h = n // 2 + 1
        nout = 4 if w["call"] == "gradient" else 1
        spec = n * n * h * c
        s1 = n * n * n * r + spec
        s2 = 2 * spec
        s3 = spec + nout * spec
        s4 = nout * 2 * spec
        s5 = nout * (spec + n * n * n * r)
    else:  # real-to-real passes
        f = n * n * n * r
        s1 = s2 = s3 = s4 = s5 = 2 * f
    return [s1, s2, s3, s4, s5]


STEP_EVENT_STRIDE = 8   # per-step CUDA events are recorded on every 8th solve of the timed region
STEP_NAMES = ["S1 fast_xw_kernel<fwd>", "S2 fast_fwd2h_kernel", "S3 fast_fused2h_kernel", "S4 fast_inv2h_kernel",
              "S5 fast_xw_kernel<inv>"]


def step_names(wname):
    """the kernel behind each of the five steps for this workload"""
    if wname == "cfg4_unbounded_256_f32":
        return STEP_NAMES
    if wname == "cfg4_unbounded_256_f64":
        return ["S1 fast_xgw_kernel<fwd>", "S2 fast64_kernel<FWD>", "S3 fast64_kernel<FUSED>", "S4 fast64_kernel<INV>", "S5 fast_xgw_kernel<inv>"]
    if wname in ("cfg3_dirichlet_255_f64", "cfg3_neumann_256_f64"):
        return ["S1 fast_xgw_kernel<fwd>", "S2 fast_r2r64_kernel<FWD>", "S3 fast_r2r64_kernel<FUSED>",
                "S4 fast_r2r64_kernel<" + ("FWD" if "dirichlet" in wname else "INV") + ">", "S5 fast_xgw_kernel<inv>"]
    if wname in ("cfg2_periodic_256_f32", "cfg2_periodic_256_f32_grad"):
        return ["S1 fast_xpw_kernel<fwd>", "S2 fast_per_kernel<FWD>", "S3 fast_per_kernel<FUSED>", "S4 fast_per_kernel<INV>",
                "S5 fast_xpw_kernel<inv>"]
    if wname == "cfg2_periodic_256_f64_grad":
        return ["S1 fast_xpw64_kernel<fwd>", "S2 fast_per64_kernel<FWD>", "S3 fast_per64_kernel<FUSED,GRAD>", "S4 fast_per64_kernel<INV>", "S5 fast_xpw64_kernel<inv>"]
    if wname == "cfg5_vector_512_f32_curl":
        return ["S1 fast_x5w_kernel<fwd>", "S2 fast5_kernel<FWD>", "S3 fast5_kernel<CURL>", "S4 fast5_kernel<INV>", "S5 fast_x5w_kernel<inv>"]
    return ["S1 xfwd_kernel", "S2 spass_kernel<0>", "S3 spass_kernel<2>", "S4 spass_kernel<1>", "S5 xinv_kernel"]


# ncu-derived counts of the dominant kernels (warp instructions, packed fp32x2 instructions, DRAM bytes per launch)
# live in profiles/ncu_counts.json together with the SHA-256 of the kernel sources they were captured from.  They
# are used only while that hash matches the sources of this checkout: a changed kernel turns "issue_view" and
# "traffic" into null instead of letting them go stale silently.
ISSUE_SLOTS_PER_CLOCK = 148 * 4
def kernel_source_hash(files):
    """SHA-256 over the named kernel sources (paths relative to the repo root, in the given order)"""
    import hashlib

    hsh = hashlib.sha256()
    for name in files:
        f = ROOT / name
        if not f.exists():
            return None
        hsh.update(Path(name).name.encode())
        hsh.update(f.read_bytes())
    return hsh.hexdigest()


def ncu_counts(wname, step_index):
    """the committed ncu counts of step `step_index` of a workload (profiles/ncu_counts.json: per workload the kernel
    source files the capture was taken from, their SHA-256, and per step the counts), or None when there is no capture
    or one of those sources has changed since"""
    f = ROOT / "profiles" / "ncu_counts.json"
    if not f.exists():
        return None
    try:
        doc = json.load(open(f))
    except Exception:
        return None
    w = doc.get("workloads", {}).get(wname)
    if not w or kernel_source_hash(w.get("sources", [])) != w.get("sources_sha256"):
        return None
    c = w.get(f"S{step_index + 1}")
    if c is not None:
        c = dict(c, capture=w.get("capture"))
    return c


def issue_view(wname, dom, kernel_ms, clocks, names):
    """The dominant kernel of the default workload is bound by instruction issue, not by HBM (profiles/r02_b.md):
    besides the HBM roofline the line carries its issue-slot utilisation = (warp instructions + packed fp32x2
    instructions: a packed instruction occupies its scheduler for two cycles) / (148 SMs x 4 schedulers x the SM clock
    sampled during the timed region) / measured kernel time.  None without a capture of the current sources."""
    c = ncu_counts(wname, dom)
    if not c or not clocks or not clocks.get("sm_mhz") or "warp_instructions" not in c:
        return None
    cycles = c["warp_instructions"] + c.get("packed_fp32x2_warp_instructions", 0)
    t_peak_ms = cycles / (ISSUE_SLOTS_PER_CLOCK * clocks["sm_mhz"] * 1e6) * 1e3
    return {"bound": "alu", "kernel": names[dom], "issue_cycles_per_launch": cycles,
            "ms_at_one_warp_instruction_per_scheduler_clock": t_peak_ms, "kernel_ms": kernel_ms, "frac": t_peak_ms / kernel_ms,
            "source": f"instruction counts of {c.get('capture', 'profiles/ncu_counts.json')} (ncu source page, same kernel sources), "
                      "SM clock of this run"}


def make_input(w, rank=0):
    """Seeded synthetic source for the workload (workloads/: generators only, no method arithmetic)."""
    import workloads as W

    dt = np.float32 if w["prec"] == "f32" else np.float64
    n = w["n"]
    seed = rank_seed(w["cfg"], rank)
    if w["kind"] == "unbounded" and w["ncomp"] == 1:
        g = W.gaussian_blobs(n, seed=seed)
        return dict(f=np.ascontiguousarray(g["f"].astype(dt)), h=g["h"], faces={})
    if w["kind"] == "unbounded":
        g = W.vortex_ring(n, seed=seed)
        return dict(f=np.ascontiguousarray(g["omega"].astype(dt)), h=g["h"], faces={})
    if w["kind"] == "periodic" and w.get("ndim", 3) == 2:
        g = W.periodic2d_modes(n, seed=seed)
        return dict(f=np.ascontiguousarray(g["f"].astype(dt)), h=tuple(L / n for L in g["L"]), faces={})
    if w["kind"] == "periodic":
        g = W.periodic3d_spectrum(n, seed=seed)
        return dict(f=np.ascontiguousarray(g["f"].astype(dt)), h=tuple(L / n for L in g["L"]), faces={})
    if w["kind"] == "dirichlet":
        g = W.dirichlet3d_manufactured(nc=n + 1, seed=seed)
    else:
        g = W.neumann3d_manufactured(nc=n, seed=seed)
    return dict(f=np.ascontiguousarray(g["f"].astype(dt)), h=g["h"],
                faces={k: np.ascontiguousarray(v.astype(dt)) for k, v in g["faces"].items()})


# ---------------------------------------------------------------------------------------- clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU through NVML while the timed region runs."""

    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
               0x80: "hw_power_brake_slowdown"}

    def __init__(self, index, period=0.004):
        super().__init__(daemon=True)
        self.period = period
        self.samples = []  # (t, sm_mhz, reasons bitmask)
        self.stop_flag = False
        self.ok = False
        try:
            import pynvml

            self.nv = pynvml
            pynvml.nvmlInit()
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # no NVML: the JSON line says so
            self.err = repr(e)
            self.max_mhz = None

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self.stop_flag:
            try:
                mhz = int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    rs = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    rs = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                self.samples.append((time.perf_counter(), mhz, rs))
            except Exception:
                pass
            time.sleep(self.period)

    def summary(self, t0, t1):
        inside = [s for s in self.samples if t0 <= s[0] <= t1]
        where = "timed region"
        if not inside:  # region shorter than one NVML query: use the nearest samples under load
            inside = sorted(self.samples, key=lambda s: min(abs(s[0] - t0), abs(s[0] - t1)))[:3]
            where = "nearest samples (timed region shorter than one NVML query)"
        if not inside:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0,
                    "note": getattr(self, "err", "no samples")}
        bits = 0
        for s in inside:
            bits |= s[2]
        reasons = [name for bit, name in self.REASONS.items() if bits & bit]
        return {"sm_mhz": float(np.median([s[1] for s in inside])), "sm_max_mhz": self.max_mhz, "reasons": reasons,
                "samples": len(inside), "where": where}


# ---------------------------------------------------------------------------------------- ncu traffic
def ncu_traffic(workload, step_index):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the dominant kernel from the committed
    ncu --set full capture of the current kernel sources (profiles/ncu_counts.json); None otherwise."""
    c = ncu_counts(workload, step_index)
    if not c or "dram_read_bytes" not in c:
        return None
    return float(c["dram_read_bytes"]) + float(c["dram_write_bytes"])


def load_peaks():
    f = ROOT / "MEASURED_PEAKS.json"
    if f.exists():
        try:
            return float(json.load(open(f))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---------------------------------------------------------------------------------------- reference arm
def oracle_solve_timer(n_sample, prec="f32"):
    """Returns (callable running ONE oracle solve of the cfg-4 workload at n_sample^3 -> (2 n_sample)^3,
    threads).  The Green's spectrum is precomputed outside the timed call."""
    import oracle as O
    import workloads as W

    g = W.gaussian_blobs(n_sample)
    f = g["f"].astype(np.float32).astype(np.float64) if prec == "f32" else g["f"]
    ghat = O.unbounded_green(g["n"], g["h"], 2.0 * g["h"][0])

    def run():
        return O.unbounded_solve(f, g["h"], ghat)

    return run, O.num_threads()


def pick_oracle_sample(budget_s, calls):
    """Largest of 64^3 / 128^3 / 256^3 whose `calls` solves fit in budget_s (calibrated on 64^3)."""
    run, _ = oracle_solve_timer(64)
    run()
    t0 = time.perf_counter()
    run()
    t64 = time.perf_counter() - t0
    n = 64
    for cand, factor in ((128, 9.5), (256, 9.5 * 9.5)):
        if t64 * factor * calls <= budget_s:
            n = cand
    return n


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    steps = args.steps if args.steps is not None else 3
    warmup = args.warmup if args.warmup is not None else 1
    n_s = pick_oracle_sample(150.0, steps + warmup)
    run, threads = oracle_solve_timer(n_s)
    for _ in range(warmup):
        run()
    t0 = time.perf_counter()
    for _ in range(steps):
        run()
    dt = (time.perf_counter() - t0) / max(steps, 1)
    value = n_s ** 3 / dt
    sample = (f"cfg-4 workload at {n_s}^3 padded to {2 * n_s}^3 (fp64 oracle, full doubled domain, "
              f"Green's spectrum precompute excluded), {steps} solves")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        # the same keys as the line of our own arm (the workload is the same; the sample of it that is timed is stated)
        "config": {"workload": DEFAULT_WORKLOAD, "grid": "256^3 padded to 512^3", "call": "sf_solve", "ncomp": 1,
                   "parallelism": "replicas x1", "l2": "host run: not applicable",
                   "timed_region": "the oracle's solve on the host cores, Green's spectrum precomputed outside (PAPER.md:53, :344); " + sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def cpu_baseline(wname=DEFAULT_WORKLOAD):
    """The oracle as it stands on the host cores, on a bounded sample of the workload: cfg 4 one full-size solve
    if it is predicted to take under ~40 s (else the 128^3 -> 256^3 copy); the other workloads one call of the
    oracle routine the parity tests compare with, at a size that keeps it to seconds."""
    import oracle as O

    w = WORKLOADS[wname]
    if wname == DEFAULT_WORKLOAD:
        n_s = pick_oracle_sample(40.0, 2)
        run, threads = oracle_solve_timer(n_s)
        what = f"1 solve of the cfg-4 workload at {n_s}^3 padded to {2 * n_s}^3, fp64 oracle on the full doubled domain, " \
               "Green's spectrum precompute excluded"
        npts = n_s ** 3
    else:
        ndim = w.get("ndim", 3)
        # direct O(N^2) sums per pencil for the real-to-real rows, recursive FFTs elsewhere: sizes chosen for seconds
        n_s = {"periodic": min(w["n"], 256), "dirichlet": 127, "neumann": 128, "unbounded": min(w["n"], 128)}[w["kind"]]
        ws = dict(w, n=n_s)
        inp = make_input(ws, 0)
        f = inp["f"].astype(np.float64)
        if w["kind"] == "periodic":
            L = tuple(hh * n_s for hh in inp["h"])
            run = lambda: O.periodic(f, L, want_grad=(w["call"] == "gradient"))
        elif w["kind"] == "dirichlet":
            run = lambda: O.dirichlet_regular(f, inp["h"], faces=inp["faces"])
        elif w["kind"] == "neumann":
            run = lambda: O.neumann_staggered(f, inp["h"], faces=inp["faces"])
        else:
            gh = O.unbounded_green((n_s,) * 3, inp["h"], 2.0 * inp["h"][0])
            rs = -1.0 if w["call"] == "curl" else 1.0
            run = lambda: O.unbounded_solve(f, inp["h"], gh, rhs_sign=rs, want_curl=(w["call"] == "curl"))
        threads = O.num_threads()
        what = f"1 call of the oracle routine of this workload ({w['kind']}, sf_{w['call']}) at {n_s}^{ndim}, fp64"
        npts = n_s ** ndim
    run()  # page in
    t0 = time.perf_counter()
    run()
    dt = time.perf_counter() - t0
    return {"value": npts / dt, "unit": UNIT, "cores": threads, "kind": "oracle", "seconds": dt, "sample": what}


# ---------------------------------------------------------------------------------------- our arm
def rank_seed(cfg, rank):
    """Every rank solves its own independent problem (replicas only): one seed per rank."""
    import workloads as W

    return W.seed_for(cfg) + 7919 * int(rank)


def max_over_ranks(values, world, device):
    """Multi-GPU timings are the max over ranks (the only collective of the bench; none on the data path)."""
    import torch
    import torch.distributed as dist

    tt = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return [float(v) for v in tt.cpu()]


def run_tc_probe():
    """one radix-16 stage of the 256-point transform as butterflies (variant 0), as a 3 x TF32
    tcgen05.mma (variant 1) and as a single TF32 product (variant 2); same data, same kernel body around the stage."""
    import torch

    import paper_2301_01145_b200 as sf

    tiles, reps = 148 * 2 * 8, 64
    g = torch.Generator(device="cuda").manual_seed(1)
    src = torch.randn((tiles, 16, 512, 2), generator=g, device="cuda", dtype=torch.float32)
    dst = torch.empty_like(src)
    ref = None
    out = {"probe": "sf_probe_dft16_stage", "tiles": tiles, "stages_per_tile": reps, "variants": {}}
    for variant, name in ((0, "fp32 pipe: exchange + radix-16 butterflies"), (1, "tcgen05.mma kind::tf32, 3 x TF32 split"),
                          (2, "tcgen05.mma kind::tf32, single product")):
        ms = min(sf.sf_probe_dft16_stage(variant, reps, tiles, src, dst) for _ in range(5))
        res = dst.double()
        if ref is None:
            ref = res.clone()
        err = float((res - ref).norm() / ref.norm())
        out["variants"][str(variant)] = {"what": name, "ms": ms, "ns_per_tile_stage_per_sm": ms * 1e6 * 148 / (tiles * reps),
                                         "rel_l2_vs_variant_0": err}
    print(json.dumps(out), flush=True)
    return 0


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2301_01145_b200 as sf

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    steps = args.steps if args.steps is not None else 200
    warmup = max(args.warmup if args.warmup is not None else 10, 3)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the hot path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    wname = args.workload
    w = WORKLOADS[wname]
    n, ncomp = w["n"], w["ncomp"]
    inp = make_input(w, rank)
    tdt = torch.float32 if w["prec"] == "f32" else torch.float64
    stream = torch.cuda.Stream()
    bc = {"unbounded": sf.SF_BC_UNBOUNDED, "periodic": sf.SF_BC_PERIODIC, "dirichlet": sf.SF_BC_DIRICHLET,
          "neumann": sf.SF_BC_NEUMANN}[w["kind"]]
    op = {"unbounded": sf.SF_OP_GREEN_GAUSS2, "periodic": sf.SF_OP_PSEUDO_SPECTRAL, "dirichlet": sf.SF_OP_FD2,
          "neumann": sf.SF_OP_FD2}[w["kind"]]
    grid = sf.SF_GRID_CELL_BOUNDARY if w["kind"] == "dirichlet" else sf.SF_GRID_CELL_CENTRE
    ndim = w.get("ndim", 3)
    plan = sf.sf_plan_create([n] * ndim, inp["h"], bc, grid=grid, op=op, prec=sf.SF_F32 if w["prec"] == "f32" else sf.SF_F64,
                             ncomp=ncomp, stream=stream.cuda_stream, rhs_sign=-1.0 if w["call"] == "curl" else 1.0)
    call = {"solve": sf.sf_solve, "gradient": sf.sf_gradient, "curl": sf.sf_curl}[w["call"]]
    out_field = sf.SF_OUT_CURL if w["call"] == "curl" else sf.SF_OUT_PSI

    # inputs resident in HBM before the timed region
    src_host = torch.from_numpy(inp["f"]).pin_memory()
    src_dev = src_host.to("cuda", non_blocking=False)
    keep = []
    for (axis, side), g in inp["faces"].items():
        t = torch.from_numpy(g).cuda()
        keep.append(t)
        sf.sf_set_bc_values(plan, axis, side, t)
    sf.sf_set_source(plan, src_dev)
    torch.cuda.synchronize()

    # ---- warm-up
    for _ in range(warmup):
        call(plan)
    sf.sf_synchronize(plan)
    launches_per_step = sf.sf_last_launch_count(plan)

    # ---- timed region: K steps, CUDA events on the plan's stream (the stream the kernels run on),
    # per-step events of the library enabled so the dominant kernel's duration is measured live
    # (every STEP_EVENT_STRIDE-th step: the five extra event records cost a few microseconds per solve)
    sf.sf_enable_step_timing(plan, min(steps, 4096))
    sf.sf_set_step_timing_stride(plan, STEP_EVENT_STRIDE if steps >= 2 * STEP_EVENT_STRIDE else 1)
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_start = time.perf_counter()
    with torch.cuda.stream(stream):
        e0.record(stream)
        for _ in range(steps):
            call(plan)
        e1.record(stream)
    barrier()
    t_end = time.perf_counter()
    sampler.stop_flag = True
    total_ms = e0.elapsed_time(e1)
    step_ms = sf.sf_step_times_ms(plan)
    sf.sf_enable_step_timing(plan, 0)
    sf.sf_set_step_timing_stride(plan, 1)
    clocks = sampler.summary(t_start, t_end)

    # ---- the same K steps without the library's inner events (cross-check of the event overhead)
    barrier()
    with torch.cuda.stream(stream):
        e0.record(stream)
        for _ in range(steps):
            call(plan)
        e1.record(stream)
    barrier()
    total_ms_noev = e0.elapsed_time(e1)

    # ---- end to end through the public API with HOST buffers: H2D of the source, solve, D2H of the
    # result, every step, inside the timed region.  The plan's copy pipeline (sf_set_pipeline, depth 2) runs the
    # upload of step k+1, the solve of step k and the download of step k-1 side by side; every step still uploads
    # its source and downloads its whole result (gradient: all 1 + ndim fields).
    nfields_out = ncomp if w["call"] != "gradient" else 1 + ndim
    fields = [(out_field, c) for c in range(ncomp)] if w["call"] != "gradient" else \
        [(sf.SF_OUT_PSI, 0)] + [(sf.SF_OUT_GRAD, a) for a in range(ndim)]
    dst_host = [torch.empty((nfields_out,) + (n,) * ndim, dtype=tdt).pin_memory() for _ in range(2)]
    e2e_steps = max(3, min(steps, 20))
    sf.sf_set_pipeline(plan, 2)

    def e2e_step(k):
        sf.sf_set_source(plan, src_host)
        call(plan)
        for i, (fld, c) in enumerate(fields):
            sf.sf_get_output_async(plan, fld, c, dst_host[k & 1][i])

    for k in range(2):
        e2e_step(k)
    sf.sf_synchronize(plan)
    barrier()
    with torch.cuda.stream(stream):
        e0.record(stream)
    for k in range(e2e_steps):
        e2e_step(k)
    sf.sf_pipeline_join(plan)      # the plan's stream waits for the copies: e1 below completes after the last download
    with torch.cuda.stream(stream):
        e1.record(stream)
    barrier()
    e2e_ms = e0.elapsed_time(e1) / e2e_steps
    # the unpipelined sequence (blocking sf_get_output on the plan's single stream), for comparison
    sf.sf_set_pipeline(plan, 1)
    barrier()
    with torch.cuda.stream(stream):
        e0.record(stream)
    for k in range(e2e_steps):
        sf.sf_set_source(plan, src_host)
        call(plan)
        for i, (fld, c) in enumerate(fields):
            sf.sf_get_output(plan, fld, c, dst_host[0][i])
    with torch.cuda.stream(stream):
        e1.record(stream)
    barrier()
    e2e_serial_ms = e0.elapsed_time(e1) / e2e_steps
    dst_host = dst_host[(e2e_steps - 1) & 1]
    h2d = src_host.numel() * src_host.element_size()
    d2h = dst_host.numel() * dst_host.element_size()
    checksum = float(dst_host.double().abs().mean())
    sf.sf_set_source(plan, src_dev)

    # ---- max over ranks
    total_ms, total_ms_noev, e2e_ms = max_over_ranks([total_ms, total_ms_noev, e2e_ms], world, "cuda")
    dev_bytes = sf.sf_device_bytes(plan)
    sf.sf_plan_destroy(plan)

    if rank == 0:
        ms_per_step = total_ms / steps
        pts = float(n) ** ndim * world
        mb = model_bytes(w)
        peak, peak_src = load_peaks()
        dom = int(np.argmax(step_ms))
        names = step_names(wname)
        ach = mb[dom] / (step_ms[dom] * 1e-3) / 1e9
        traffic = ncu_traffic(wname, dom)
        line = {
            "metric": METRIC, "value": pts / (ms_per_step * 1e-3), "unit": UNIT, "n_gpus": world, "steps": steps,
            "warmup": warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": w["prec"], "data": "synthetic",
            "config": {"workload": wname, "grid": f"{n}^{ndim}" + (f" padded to {2 * n}^{ndim}" if w["kind"] == "unbounded" else ""),
                       "call": "sf_" + w["call"], "ncomp": ncomp, "parallelism": f"replicas x{world}",
                       "l2": ("no flush needed: every step streams its whole working set through HBM "
                              f"({sum(mb) / 1e6:.0f} MB algorithmic per step, plan holds {dev_bytes / 1e6:.0f} MB) >> 126 MB L2")
                             if sum(mb) > 4 * 126e6 else
                             (f"not flushed: the working set ({sum(mb) / 1e6:.1f} MB algorithmic per step) is of the order of / below the "
                              "126 MB L2, so part of every pass is served from L2; the roofline fraction of this "
                              "workload is not an HBM statement"),
                       "timed_region": "sf_solve x K back to back, source and output resident in HBM, Green's spectrum "
                                       "precomputed at plan time (PAPER.md:53, :344)"},
            "clocks": clocks,
            "e2e": {"value": pts / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "steps": e2e_steps, "result_checksum_mean_abs": checksum,
                    "ms_per_step_single_stream": e2e_serial_ms,
                    "path": "sf_set_pipeline(2); per step: sf_set_source(pinned host) -> sf_" + w["call"] + " -> sf_get_output_async(pinned host), "
                            "every field of the result; upload, compute and download of neighbouring steps overlap; "
                            "timed with CUDA events on the plan's stream, the end event behind sf_pipeline_join"},
            "gpu_launches": launches_per_step * steps,
            "roofline": {"bound": "hbm", "kernel": names[dom], "achieved": ach, "peak": peak, "unit": "GB/s",
                         "frac": ach / peak, "traffic": traffic, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": mb[dom], "kernel_ms": step_ms[dom]},
            "steps_ms": {names[i]: step_ms[i] for i in range(5)},
            "steps_ms_note": "CUDA events of the library around each of the five launches, on every "
                             f"{STEP_EVENT_STRIDE if steps >= 2 * STEP_EVENT_STRIDE else 1}-th step of the timed region; "
                             "their sum exceeds ms_per_step by the cost of the event records themselves",
            "issue_view": issue_view(wname, dom, step_ms[dom], clocks, names),
            "steps_gbs": {names[i]: (mb[i] / (step_ms[i] * 1e-3) / 1e9 if step_ms[i] > 0 else None) for i in range(5)},
            "solve_roofline": {"algorithmic_bytes_per_step": sum(mb), "achieved_gbs": sum(mb) / (ms_per_step * 1e-3) / 1e9,
                               "frac_of_measured_peak": sum(mb) / (ms_per_step * 1e-3) / 1e9 / peak,
                               "frac_of_8TBs_nominal": sum(mb) / (ms_per_step * 1e-3) / 1e9 / 8000.0},
            "ms_per_step_without_step_events": total_ms_noev / steps,
            "step_event_stride": STEP_EVENT_STRIDE if steps >= 2 * STEP_EVENT_STRIDE else 1,
        }
        if world == 1 and not args.no_cpu_baseline and wname == DEFAULT_WORKLOAD:   # the oracle sample is the cfg-4 workload
            line["cpu_baseline"] = cpu_baseline(wname)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--tc-probe", action="store_true",
                    help="time the radix-16 exchange + DFT stage on the fp32 pipe and on the tensor cores (sf_probe_dft16_stage) and exit")
    args = ap.parse_args()
    if args.tc_probe:
        return run_tc_probe()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
