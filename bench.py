#!/usr/bin/env python
"""bench.py — throughput of the hydrostatic free-surface time step (libocn) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

One "step" is one baroclinic time step = the whole hot path over the
seeded synthetic workload of BASELINE.json config C (default 4: 2880x1200x100 near-global
lat-lon grid, fp32, 40 barotropic sub-steps — the configuration the metric is quoted on).
Prints ONE JSON line (rank 0): cell-updates/s (all grid cells, land included — the paper's
"grid size" convention), SYPD-equivalent, per-stage device times, the HBM
roofline of the dominant kernel, the end-to-end number through the C ABI with host buffers,
and the CPU oracle timed on this box's host cores as a reported baseline.

N > 1 (torchrun): the path does not shard in this round ("replicas only"): every
rank steps an independent replica of the same workload on its own GPU, no data-path collective;
time = max over ranks, value = N x cells x K / time, scaling "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "cell_updates_per_s"
UNIT = "cell-updates/s"
# algorithmic HBM bytes per wet cell-update of each stage: compulsory reads + writes; every array is
# `word` bytes per value except the hydrostatic pressure, which is stored in fp64 in both precisions
# With the Ri closure (--closure ri) K1 evaluates (nu, kappa) on chip and writes the 3 modified
# super-diagonals of the per-column solves, which K3 reads: + 3 words each.
# algorithmic floating-point operations of K1 per wet cell-update (+, -, x, / of the formulas of sections
# 3.4-3.8 as written, every face reconstructed once, all orders 3): 8 WENO reconstructions x 68 + fluxes and divergence 56 +
# zeta, K, D 24 + the u and v points 86 + quasi-AB2, predictor, elimination, column sums, w 42
K1_FLOPS_PER_WET_CELL = 8 * 68 + 56 + 24 + 86 + 42


def stage_bytes(stage, word, closure=0):
    b = {"tendency": (16 + (3 if closure else 0)) * word + 8, "backsub_correct_pressure": (8 + (3 if closure else 0)) * word + 8}
    return b.get(stage)
# window of config 4 the oracle is timed on: (j0, j1, i0, i1)
CPU_WINDOW = (500, 700, 1300, 1700)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--closure", default="const", choices=["const", "ri"],
                    help="vertical mixing: constant coefficients (default, the north_star path) or the Ri-based closure "
                         "of PAPER.md:114 (SURVEY 8f-1; DESIGN.md §3.12)")
    ap.add_argument("--patch", default="16x4", help="config 6 only (kernel analysis): WxH ocean patch of every 32x8 tile")
    ap.add_argument("--bands", type=int, default=0,
                    help="(analysis, DESIGN.md section 9) step the grid as this many latitude bands: all on this one GPU "
                         "(no torchrun: time of the slowest-possible serial execution / N = the projected band time), "
                         "or one band per rank under torchrun with --gpus N (strong scaling, NCCL point-to-point)")
    ap.add_argument("--fused-put", action="store_true",
                    help="with --bands: the back-substitution kernel stores the 3-D overlap rows into the neighbours' arrays itself "
                         "(peer memory; CUDA IPC under torchrun) instead of packing and sending them")
    ap.add_argument("--ny", type=int, default=0,
                    help="with --bands: rows of the whole grid instead of the configuration's (weak-scaling projection: "
                         "--config 5 --ny 1800 --bands 2 gives every band the 900 rows of the aqua-planet)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the end-to-end (host buffer) leg")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-closure-leg", action="store_true", help="skip the second model with the Ri closure")
    return ap.parse_args()


def workload_name(wl):
    g = wl["grid"]
    return "%s %dx%dx%d fp%d M=%d dt=%gs" % (wl["name"], g["nx"], g["ny"], g["nz"], wl["params"]["precision"],
                                             wl["params"]["substeps"], wl["params"]["dt"])


def sypd(dt, sec_per_step):
    return dt / (365.0 * sec_per_step)          # the paper's year is 365 d


# ---------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline and --impl reference)
# ---------------------------------------------------------------------------------------------
def oracle_sample(config, closure="const"):
    from paper_2309_06662_b200 import workloads as W
    wl, what = _oracle_sample(config)
    if closure == "ri":
        W.with_ri_closure(wl)
        what += ", Ri closure"
    return wl, what


def _oracle_sample(config):
    from paper_2309_06662_b200 import workloads as W
    if config == 4:
        wl = W.config4(window=CPU_WINDOW, steps=1)
        what = "config 4 window j=%d:%d i=%d:%d (closed box, identical physics)" % CPU_WINDOW
    elif config == 5:
        wl = W.aquaplanet(window=(300, 500, 900, 1300), steps=1)
        what = "aqua-planet window j=300:500 i=900:1300 (closed box)"
    elif config == 6:
        wl = W.make(6, nx=320, ny=160)
        what = "patch planet 320x160 (default patch)"
    elif config in (2, 3):
        wl = W.make(config, window=(200, 400, 500, 900), steps=1)
        what = "config %d window j=200:400 i=500:900 (closed box)" % config
    else:
        wl = W.make(config)
        what = "config %d full size" % config
    return wl, what


def time_oracle(config, steps, warmup, closure="const", threads=None, shrink=False):
    import oracle
    oracle.build()
    if threads:
        oracle.set_num_threads(threads)
    wl, what = oracle_sample(config, closure)
    if shrink and config == 4:                   # the 1-thread figure: a quarter of the window, same physics
        from paper_2309_06662_b200 import workloads as W
        wl = W.config4(window=(500, 600, 1300, 1500), steps=1)
        what = "config 4 window j=500:600 i=1300:1500 (closed box, identical physics)"
        if closure == "ri":
            W.with_ri_closure(wl)
    g = wl["grid"]
    cells = g["nx"] * g["ny"] * g["nz"]
    ref = oracle.RefModel(wl)
    nwet = int(ref.grid.masks()["wet"].sum(dtype=np.int64))
    ref.step(max(1, warmup))                     # Euler start + AB2 warm-up
    t0 = time.perf_counter()
    ref.step(steps)
    dt = time.perf_counter() - t0
    return dict(value=cells * steps / dt, wet_value=nwet * steps / dt, wet_fraction=nwet / cells,
                sec_per_step=dt / steps, cores=oracle.num_threads(), cells=cells,
                sample="%s: %dx%dx%d cells, %d steps after %d warm-up" % (what, g["nx"], g["ny"], g["nz"], steps,
                                                                         max(1, warmup)),
                dt_model=wl["params"]["dt"], name=workload_name(wl))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    steps = min(args.steps, 3) if args.config >= 2 else args.steps
    r = time_oracle(args.config, steps, min(args.warmup, 2), args.closure)
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": min(args.warmup, 2), "ms_per_step": 1e3 * r["sec_per_step"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": r["name"], "sample": r["sample"]},
            "sypd_equivalent_of_sample": sypd(r["dt_model"], r["sec_per_step"]),
            "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle",
                             "sample": r["sample"], "wet_cell_updates_per_s": r["wet_value"],
                             "wet_fraction_of_sample": r["wet_fraction"]},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md recipe)
# ---------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, device):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(device), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            pass

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.f.read().splitlines():
            c = [x.strip() for x in ln.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2]))
            except ValueError:
                continue
            for n, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_entry(workload, kernel):
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            e = json.load(f).get(kernel + ("+ri" if "+ri" in workload else ""))
        return e if e and e.get("workload") == workload else None
    except Exception:
        return None


def ncu_step_traffic(workload):
    """DRAM bytes of one whole step (all kernels) from the committed ncu capture of this workload, if any."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            e = json.load(f).get("step" + ("+ri" if "+ri" in workload else ""))
        return float(e["dram_bytes_per_step"]) if e and e.get("workload") == workload else None
    except Exception:
        return None


def ncu_traffic(workload, kernel):
    """DRAM bytes per launch of `kernel` from the committed ncu --set full capture, if it was taken
    on this workload (profiles/traffic.json, written by hand from the capture's raw page)."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            t = json.load(f)
        e = t.get(kernel + ("+ri" if "+ri" in workload else ""))
        if e and e.get("workload") == workload:
            return float(e["dram_bytes_per_launch"])
    except Exception:
        pass
    return None


# ---------------------------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------------------------
def wet_cells(model):
    import ctypes as C
    from paper_2309_06662_b200 import ocn
    wet = np.zeros((model.nz, model.ny, model.nx), np.uint8)
    rc = ocn.lib().ocn_get_masks(model.grid.h, C.c_void_p(wet.ctypes.data), None, None, None, None, None)
    assert rc == 0
    return int(wet.sum(dtype=np.int64))


def run_ours(args):
    import torch
    from paper_2309_06662_b200 import build as ocn_build
    from paper_2309_06662_b200 import ocn, replicas, workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libocn has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        ocn_build.build()
    if dist is not None:
        dist.barrier()

    K, Wm = args.steps, max(args.warmup, 3)
    if args.config == 6:
        pw, ph = (int(x) for x in args.patch.lower().split("x"))
        wl = W.make(6, w=pw, h=ph)
    else:
        wl = W.make(args.config)
    if args.closure == "ri":
        W.with_ri_closure(wl)
    ri = 1 if args.closure == "ri" else 0
    g, prm = wl["grid"], wl["params"]
    nx, ny, nz = g["nx"], g["ny"], g["nz"]
    cells = nx * ny * nz
    np_dtype = np.float32 if prm["precision"] == 32 else np.float64
    t_dtype = torch.float32 if prm["precision"] == 32 else torch.float64
    stream = torch.cuda.Stream(device=local)
    model = ocn.Model(wl, device=local, stream=stream.cuda_stream)
    nwet = wet_cells(model)
    info = model.info()

    def barrier():
        replicas.barrier(dist, torch.cuda.synchronize)

    def max_over_ranks(x):
        return replicas.max_over_ranks(x, dist, device="cuda")

    # ---- device-resident timing: K steps of the production path (one CUDA graph launch per step) ----
    clocks = ClockSampler(local)                 # samples from the warm-up on: nvidia-smi needs ~0.2 s to start
    model.time_step(Wm)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    model.time_step(K)
    e1.record(stream)
    barrier()
    ms_total = max_over_ranks(e0.elapsed_time(e1))
    # ---- same K steps again with an event between stages: per-kernel durations for the roofline ----
    model.profile_enable(True)
    model.time_step(1)
    model.profile_read(reset=True)
    model.time_step(K)
    stages = model.profile_read(reset=True)
    model.profile_enable(False)
    clk = clocks.stop()
    sec_per_step = ms_total * 1e-3 / K
    value = replicas.aggregate_throughput(cells, K, ms_total, world)

    # finite check of the state the timed steps produced (d2h of eta only)
    eta = model.get_fields(names=("eta",))["eta"]
    assert np.isfinite(eta).all(), "non-finite eta after the timed steps"

    # ---- roofline of the dominant kernel ----
    peak, peak_src = measured_peak()
    word = 4 if prm["precision"] == 32 else 8
    dom = max(stages, key=lambda s: stages[s]["ms"])
    dom_bytes = stage_bytes(dom, word, ri)
    roof = None
    stage_out = {}
    for s, v in stages.items():
        stage_out[s] = {"ms_per_step": v["ms"] / K, "launches_per_step": v["launches"] / K}
        if stage_bytes(s, word, ri) and v["launches"]:
            stage_out[s]["algorithmic_gbs"] = stage_bytes(s, word, ri) * nwet / (v["ms"] / K * 1e-3) / 1e9
    if dom_bytes is not None:
        alg_bytes = dom_bytes * nwet
        ach = alg_bytes / (stages[dom]["ms"] / K * 1e-3) / 1e9
        roof = {"kernel": dom, "bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes,
                "bytes_per_wet_cell": dom_bytes, "traffic": ncu_traffic(workload_name(wl), dom)}
    else:                       # the 2-D sub-cycle dominates (tiny 3-D grids): 16 words per column per sub-step
        ncol = nx * ny
        alg_bytes = 16 * word * ncol * prm["substeps"]
        ach = alg_bytes / (stages[dom]["ms"] / K * 1e-3) / 1e9
        roof = {"kernel": dom, "bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes, "traffic": None}

    # K1 is bound by instruction issue, not by HBM.  This is an issue-slot UTILISATION (all executed warp
    # instructions, integer and control included, of the committed ncu capture against 148 SMs x 4 schedulers x SM clock),
    # not a roofline of useful work
    issue_util = None
    ent = ncu_entry(workload_name(wl), dom)
    if ent and "warp_instructions_per_launch" in ent:
        mhz = clk.get("sm_mhz") or 1965.0
        slots = 148 * 4 * mhz * 1e6 * (stages[dom]["ms"] / K * 1e-3)
        issue_util = {"kernel": dom, "warp_instructions_per_launch": ent["warp_instructions_per_launch"],
                      "issue_slots_per_launch": slots, "utilisation": ent["warp_instructions_per_launch"] / slots,
                      "source": "profiles/traffic.json (ncu smsp__inst_executed.sum) / (148 SMs x 4 schedulers x sampled SM clock x live K1 time)"}
    # second view of K1, which is bound by arithmetic: the flops of the formulas as written (NOT executed instructions) against
    # the plain-ALU peak of the chip, 148 SMs x 128 fp32 lanes (64 in fp64) x 2 flop per FMA x sampled SM clock
    roof_alu = None
    if dom == "tendency":
        mhz = clk.get("sm_mhz") or 1965.0
        peak_tf = 148 * (128 if word == 4 else 64) * 2 * mhz * 1e6 / 1e12
        ach_tf = K1_FLOPS_PER_WET_CELL * nwet / (stages[dom]["ms"] / K * 1e-3) / 1e12
        roof_alu = {"kernel": dom, "bound": "alu", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach_tf / peak_tf,
                    "flops_per_wet_cell": K1_FLOPS_PER_WET_CELL,
                    "peak_source": "148 SMs x %d lanes x 2 (FMA) x sampled SM clock; flop count of the formulas: DESIGN.md section 7"
                                   % (128 if word == 4 else 64)}
    # the whole step against the HBM roofline (north_star's target is 0.60 for the fused step on config 4)
    step_bytes = sum((stage_bytes(s_, word, ri) or 0) for s_ in stages) * nwet + 16 * word * nx * ny * (info["launches_per_step"] - 3)
    roof_step = {"bound": "hbm", "algorithmic_bytes_per_step": step_bytes, "achieved": step_bytes / sec_per_step / 1e9,
                 "peak": peak, "unit": "GB/s", "frac": step_bytes / sec_per_step / 1e9 / peak, "target_frac": 0.60,
                 "what": "per wet cell: K1 %d B + K3 %d B; barotropic: 16 words per column per resident group of sub-steps (%d groups)"
                         % (stage_bytes("tendency", word, ri), stage_bytes("backsub_correct_pressure", word, ri), info["launches_per_step"] - 3)}
    tr = ncu_step_traffic(workload_name(wl))
    if tr:
        roof_step.update({"traffic": tr, "traffic_gbs": tr / sec_per_step / 1e9, "traffic_frac": tr / sec_per_step / 1e9 / peak})

    # ---- end to end through the C ABI with HOST (pinned) buffers ----
    # e2e: every step copies that step's forcing (tau_x, tau_y) host -> device and reads that step's result (eta) device ->
    # host, through the public calls a user makes; the read-back is left in flight (ocn_get_fields_async) and waited for one
    # step later, so that step n + 1 is enqueued while the result of step n travels.  The initial state is uploaded before
    # the timed region (an initial condition, like weights).  e2e_with_state_io is round 1's definition: it adds the upload
    # of the full state and the download of the full state + w to the timed region, amortised over the steps (PCIe bound).
    e2e = e2e_state = None
    if not args.no_e2e:
        f = wl["fields"]
        pin = {k: torch.from_numpy(np.ascontiguousarray(f[k], dtype=np_dtype)).pin_memory()
               for k in ("u", "v", "T", "S", "eta", "tau_x", "tau_y")}
        out = {k: torch.empty(pin[k].shape, dtype=t_dtype).pin_memory() for k in ("u", "v", "T", "S", "eta")}
        out["w"] = torch.empty((nz + 1, ny, nx), dtype=t_dtype).pin_memory()
        eta_step = [torch.empty((ny, nx), dtype=t_dtype).pin_memory() for _ in range(2)]
        Ke = K
        b2 = ny * nx * word
        checks = []

        def steps_job():
            tickets = []
            for n in range(Ke):
                model.set_fields_ptr(tau_x=pin["tau_x"].data_ptr(), tau_y=pin["tau_y"].data_ptr())   # this step's forcing
                model.time_step(1)
                tickets.append(model.get_fields_async_ptr(eta=eta_step[n % 2].data_ptr()))            # this step's result
                if n >= 1:
                    model.wait(tickets[n - 1])
                    checks.append(float(eta_step[(n - 1) % 2][ny // 2, nx // 2]))                   # the host consumes it
            model.wait(tickets[-1])
            checks.append(float(eta_step[(Ke - 1) % 2][ny // 2, nx // 2]))

        def state_job():
            model.set_fields_ptr(**{k: pin[k].data_ptr() for k in ("u", "v", "T", "S", "eta", "tau_x", "tau_y")})
            steps_job()
            model.get_fields_ptr(**{k: out[k].data_ptr() for k in out})

        def timed(job):
            barrier()
            t0 = time.perf_counter()
            job()
            model.synchronize()
            barrier()
            return max_over_ranks((time.perf_counter() - t0) * 1e3)        # host wall clock around the public calls

        state_job()                                 # warm-up (also re-creates the AB2 start)
        ms_s = timed(state_job)
        ms_e = timed(steps_job)
        assert all(np.isfinite(c) for c in checks)
        e2e = {"value": world * cells * Ke / (ms_e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 2 * b2,
               "d2h_bytes_per_step": b2, "steps": Ke, "ms_per_step": ms_e / Ke,
               "what": "per step: ocn_set_fields(tau_x, tau_y; pinned host) + ocn_time_step(1) + ocn_get_fields_async(eta) "
                       "waited for one step later; host wall clock; state resident (uploaded before the timed region)"}
        e2e_state = {"value": world * cells * Ke / (ms_s * 1e-3), "unit": UNIT,
                     "h2d_bytes_per_step": (4 * cells * word + 3 * b2) / Ke + 2 * b2,
                     "d2h_bytes_per_step": (4 * cells * word + (nz + 1) * b2 + b2) / Ke + b2, "steps": Ke,
                     "what": "round 1's definition: the same plus ocn_set_fields(full state) before and ocn_get_fields(full "
                             "state + w) after the steps inside the timed region, amortised over the steps (PCIe bound)"}
        del pin, out
    model.close()

    # ---- the same workload with the Ri-based closure the paper uses in every run ----
    wname = workload_name(wl)
    closure_line = None
    if not ri and args.config >= 2 and not args.no_closure_leg:
        wlr = W.with_ri_closure(wl)
        mr = ocn.Model(wlr, device=local, stream=stream.cuda_stream)
        mr.time_step(Wm)
        barrier()
        e0.record(stream)
        mr.time_step(K)
        e1.record(stream)
        barrier()
        ms_r = max_over_ranks(e0.elapsed_time(e1))
        mr.profile_enable(True); mr.time_step(1); mr.profile_read(reset=True)
        mr.time_step(K)
        st_r = mr.profile_read(reset=True)
        mr.profile_enable(False)
        assert np.isfinite(mr.get_fields(names=("eta",))["eta"]).all()
        mr.close()
        closure_line = {"closure": "ri", "ms_per_step": ms_r / K, "value": replicas.aggregate_throughput(cells, K, ms_r, world),
                        "sypd_equivalent": sypd(prm["dt"], ms_r * 1e-3 / K),
                        "stages_ms": {s_: v["ms"] / K for s_, v in st_r.items()}}

    # ---- CPU oracle on this box's host cores (rank 0, N = 1 only) ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        r = time_oracle(args.config, 3 if args.config >= 2 else 5, 1, args.closure)
        r1 = time_oracle(args.config, 1, 1, args.closure, threads=1, shrink=True)
        cpu = {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"],
               "wet_cell_updates_per_s": r["wet_value"], "wet_fraction_of_sample": r["wet_fraction"],
               "one_thread": {"value": r1["value"], "wet_cell_updates_per_s": r1["wet_value"], "cores": 1, "sample": r1["sample"]}}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
                "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32" if prm["precision"] == 32 else "f64", "data": "synthetic",
                "config": {"workload": wname, "cells": cells, "wet_cells": nwet,
                           "l2": "working set %.1f GB >> 126 MB L2 (no flush needed)" % (info["device_bytes"] / 1e9)
                                 if info["device_bytes"] > 1e9 else "working set fits L2 (launch/latency bound; roofline n/a)",
                           "parallelism": "replicas x%d (independent ensemble members, no exchange; the sharded form of the "
                                          "path, latitude bands with one exchange step, runs with --bands N: DESIGN.md section 9)" % world},
                "sypd_equivalent": sypd(prm["dt"], sec_per_step),
                "wet_cell_updates_per_s": world * nwet * K / (ms_total * 1e-3),
                "stages": stage_out, "roofline": roof, "roofline_step": roof_step, "roofline_alu": roof_alu, "issue_utilisation": issue_util, "e2e": e2e,
                "e2e_with_state_io": e2e_state, "closure_ri": closure_line, "cpu_baseline": cpu,
                "gpu_launches": info["launches_per_step"] * K, "clocks": clk,
                "device_bytes": info["device_bytes"]}
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def run_bands(args):
    """--bands N: the grid as N latitude bands (paper_2309_06662_b200/bands.py).  Single process: all bands on this GPU, one
    stream — their summed time / N is what one GPU of N would spend on its band (kernels + packing; the copies between
    bands run at HBM instead of NVLink speed, so the line also gives the bytes per cut and their time at NVLink speed).
    Under torchrun: one band per rank, exchanges over NCCL, strong scaling of the whole grid."""
    import torch
    from paper_2309_06662_b200 import bands, build as ocn_build
    from paper_2309_06662_b200 import ocn, replicas, workloads as W

    rank, world, local = (int(os.environ.get(k, d)) for k, d in (("RANK", "0"), ("WORLD_SIZE", "1"), ("LOCAL_RANK", "0")))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libocn has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        ocn_build.build()
    if dist is not None:
        dist.barrier()
    K, Wm = args.steps, max(args.warmup, 3)
    wl = W.make(args.config, ny=args.ny) if args.ny > 0 else W.make(args.config)
    if args.closure == "ri":
        W.with_ri_closure(wl)
    g, prm = wl["grid"], wl["params"]
    cells = g["nx"] * g["ny"] * g["nz"]
    stream = torch.cuda.Stream(device=local)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def timed(obj):
        obj.time_step(Wm)
        replicas.barrier(dist, torch.cuda.synchronize)
        e0.record(stream)
        obj.time_step(K)
        e1.record(stream)
        replicas.barrier(dist, torch.cuda.synchronize)
        return replicas.max_over_ranks(e0.elapsed_time(e1), dist, device="cuda") / K

    clocks = ClockSampler(local)
    with torch.cuda.stream(stream):
        if world > 1:
            if args.bands != world:
                raise SystemExit("bench.py --bands N under torchrun: N must equal the number of ranks")
            B = bands.DistBand(wl, dist, device=local, stream=stream.cuda_stream, fused_put=args.fused_put)
            ms = timed(B)
            m0, nb, whole_ms = B.model, world, None
        else:
            whole = ocn.Model(wl, device=local, stream=stream.cuda_stream)
            whole_ms = timed(whole)
            whole.close()
            B = bands.Bands(wl, args.bands, device=local, stream=stream, fused_put=args.fused_put)
            ms = timed(B)
            m0, nb = B.models[len(B.models) // 2], args.bands
        groups = [bands.group_after_part(p, B.parts) for p in range(B.parts)]
        if args.fused_put:                               # the 3-D rows are put by the kernel: only (eta, U, V) are packed at the end
            groups = [ocn.ROWS_STATE_2D if gr == ocn.ROWS_STATE else gr for gr in groups]
        sent = {gr: m0.rows_bytes(gr, B.h) for gr in set(groups) if gr is not None}
        bytes_cut = sum(sent[gr] for gr in groups if gr is not None)
        bytes_put = m0.rows_bytes(ocn.ROWS_STATE, B.h) - m0.rows_bytes(ocn.ROWS_STATE_2D, B.h) if args.fused_put else 0
        eta_ok = bool(np.isfinite(m0.get_fields(("eta",))["eta"]).all())
    clk = clocks.stop()
    assert eta_ok, "non-finite eta after the timed steps"
    if rank == 0:
        nvl = bytes_cut / 900e9 * 1e3                   # one direction of one cut at NVLink 5 speed (both directions run at once)
        out = {"metric": METRIC, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm, "higher_is_better": True,
               "dtype": "f32" if prm["precision"] == 32 else "f64", "data": "synthetic", "vs_baseline": None, "clocks": clk,
               "config": {"workload": workload_name(wl), "cells": cells,
                          "parallelism": ("%d latitude bands, one per GPU (NCCL send / recv)" % nb) if world > 1
                                         else "%d latitude bands, ALL ON ONE GPU (projection of the band time)" % nb},
               "bands": {"n": nb, "overlap_rows": B.h, "own_rows": [o[1] - o[0] for o in B.own], "parts_per_step": B.parts,
                         "exchanges_per_step": sum(gr is not None for gr in groups),
                         "fused_put": bool(args.fused_put), "bytes_put_by_the_kernel_per_step_per_cut_and_direction": bytes_put,
                         "bytes_per_step_per_cut_and_direction": bytes_cut, "ms_of_those_bytes_at_900_GB_s": nvl}}
        if world > 1:
            out.update(value=cells * 1e3 / ms, ms_per_step=ms, scaling="strong")
        else:
            per_band = ms / nb
            out.update(value=cells * 1e3 / ms, ms_per_step=ms, scaling="n/a (one GPU)")
            out["bands"].update(ms_per_step_whole_grid_one_model=whole_ms, ms_per_step_all_bands_on_one_gpu=ms,
                                ms_per_step_per_band=per_band,
                                redundant_rows_fraction=sum(e[1] - e[0] for e in B.ext) / g["ny"] - 1.0,
                                projected_speedup_on_n_gpus=whole_ms / (per_band + nvl),
                                projected_speedup_if_the_puts_do_not_overlap=whole_ms / (per_band + nvl + bytes_put / 900e9 * 1e3))
        print(json.dumps(out))
    B.close()
    if dist is not None:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    elif args.bands > 0:
        run_bands(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
