#!/usr/bin/env python
"""bench.py -- throughput of the mphv hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl mphv|reference]

A step = one pass of the whole hot path over the workload: the full split step S_x, S_y, [S_z],
V_vx, V_vy, V_vz followed by the moments n, j, P (mphv_step_moments through the C ABI).
Metric: phase-space cell-updates/s = cells x steps / time (BASELINE.json), fp64.
N = 1 runs BASELINE.json configs[3] (2D3V 128x64x40^3, the headline roofline config).
N > 1 (torchrun): weak scaling by spatial block decomposition (the paper's own
parallelisation): the periodic x axis is N times longer, every rank owns one
configs[3]-sized block and exchanges its two boundary layers with both x neighbours before the
X stage (mphv_pack_halo -> NCCL send/recv -> mphv_stage_x_halo: S_x with the received ghost layers and S_y
in one pass); time = max over ranks.
--decomp none instead runs N independent seeded problems (no exchange); --decomp halo at N = 1
sends the spatial sweeps through the same pack / halo kernels with the block as its own neighbour.
JSON keys beyond the contract: "e2e" = mphv_run_host (f itself crosses PCIe both ways every step);
"e2e_resident" = mphv_step_fields_host (f resident; host E, B in and host n, j, P out every step).
--impl reference times the CPU oracle (oracle/) on a bounded spatial sub-block of the same
workload on the host cores; rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import numpy as np

METRIC = "phase_space_cell_updates_per_sec"
UNIT = "cell-updates/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs index (default 3, headline)")
    ap.add_argument("--impl", default="mphv", choices=["mphv", "reference"])
    ap.add_argument("--fusion", type=int, default=3, choices=[0, 1, 2, 3],
                    help="mphv_set_fusion level: 0 one kernel per sweep, 1 pairwise fused, 2 whole V stage in one kernel, 3 also S_x+S_y in one kernel; default 3")
    ap.add_argument("--vmode", default="plain", choices=["plain", "backsub"],
                    help="V stage: plain 1-D sweeps (BASELINE.json north_star, default) or backsubstitution (P:L137)")
    ap.add_argument("--decomp", default="auto", choices=["auto", "halo", "none"],
                    help="'halo' = one spatially decomposed problem with neighbour exchange (the default for N > 1; "
                         "at N = 1 the block is its own periodic neighbour), 'none' = N independent problems "
                         "(the default at N = 1)")
    ap.add_argument("--aux", action="store_true",
                    help="instead of the step: time the coupling kernels of SURVEY 8(f) (ten-moment Maxwellian fill, "
                         "exchange of Maxwellians, moment matching) on the same workload and print one JSON line")
    ap.add_argument("--no-two-species", action="store_true",
                    help="skip the coupled two-species leg (ions + electrons + Maxwell, extra key two_species)")
    ap.add_argument("--species-steps", type=int, default=6)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--cpu-seconds", type=float, default=30.0,
                    help="CPU work the oracle sample is sized for over 20 steps (estimated; about a third of it on a 16-core box)")
    return ap.parse_args()


# ------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock and throttle reasons with NVML during the timed region."""

    def __init__(self, index: int, period: float = 0.02):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self.period, self._stop, self._thr, self.h = period, threading.Event(), None, None
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception as e:  # noqa: BLE001
            self.err = repr(e)

    def _run(self):
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:  # noqa: BLE001
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:  # noqa: BLE001
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.h is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                    "note": "no NVML samples"}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------- oracle legs
def oracle_sample(w, cpu_seconds: float):
    """A spatial sub-block of workload w (same velocity grid, same f0/E/B recipe and dt rule,
    block centred on the current sheet) sized for about cpu_seconds of oracle work."""
    from paper_2305_01487_b200 import inputs
    est_rate = 1.5e7 * max(1, os.cpu_count() or 1) ** 0.7      # cell-updates/s guess, plain C oracle
    nvel = int(np.prod(w.nv))
    target_space = max(16, int(cpu_seconds * est_rate / nvel))
    if w.nx[2] > 1:
        side = int(max(4, min(w.nx[0], round(target_space ** (1 / 3)))))
        nx = (side, side, side)
    elif w.nx[1] > 1:
        sy = int(max(4, min(w.nx[1], round((target_space / 2) ** 0.5))))
        sx = int(max(4, min(w.nx[0], target_space // sy)))
        nx = (sx, sy, 1)
    else:
        nx = w.nx
    dx = [w.dx(d) for d in range(3)]
    xlo, xhi = list(w.xlo), list(w.xhi)
    for d in range(3):
        if w.nx[d] > 1:
            mid = 0.5 * (w.xlo[d] + w.xhi[d]) if d == 1 else w.xlo[d] + 0.5 * nx[d] * dx[d]
            xlo[d] = mid - 0.5 * nx[d] * dx[d]
            xhi[d] = mid + 0.5 * nx[d] * dx[d]
    sub = inputs.variant(w, name=w.name + f"_sub{nx[0]}x{nx[1]}x{nx[2]}", nx=tuple(nx),
                         xlo=tuple(xlo), xhi=tuple(xhi))
    return sub


SAMPLE_STEPS = 20          # the oracle sample is sized for cpu_seconds of work over this many steps (= the default --steps)


def time_oracle(w, steps: int, warmup: int, cpu_seconds: float):
    """Times oracle.step + oracle.moments, as they stand, on a bounded sample of workload w. ONE sample per workload:
    the cpu_baseline leg and the --impl reference arm time the same sub-block (sized for cpu_seconds / SAMPLE_STEPS of
    oracle work per step), and with default flags the same number of steps; a long reference run (steps + warmup
    above 200) shrinks the block so that the whole run stays within a few minutes."""
    import oracle
    from paper_2305_01487_b200 import inputs
    sub = oracle_sample(w, min(cpu_seconds / SAMPLE_STEPS, 150.0 / max(1, steps + warmup)))
    f0, E, B, _ = inputs.make_all(sub)
    dt = 0.5 * inputs.cfl_dt(sub, E, B)          # safely inside |s| < 1 on the sub-block
    grid, box = oracle.Grid(sub.nx, sub.nv, sub.bc), oracle.Box(sub.xlo, sub.xhi, sub.vlo, sub.vhi)
    f = f0.copy()
    for _ in range(warmup):
        oracle.step(f, grid, box, sub.q_over_m, E, B, dt)
        oracle.moments(f, grid, box)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle.step(f, grid, box, sub.q_over_m, E, B, dt)
        oracle.moments(f, grid, box)
    el = time.perf_counter() - t0
    return {
        "value": sub.n_cells * steps / el, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
        "sample": f"{sub.nx[0]}x{sub.nx[1]}x{sub.nx[2]} spatial sub-block x {sub.nv[0]}x{sub.nv[1]}x{sub.nv[2]} velocity "
                  f"({sub.n_cells} cells) of {w.name}, {steps} full split steps + moments, {el:.2f} s",
        "ms_per_step": 1e3 * el / steps,
    }


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    steps, warmup = max(1, args.steps), max(0, args.warmup)
    r = time_oracle(w, steps, warmup, args.cpu_seconds)
    line = {
        "impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "note": "CPU oracle on a bounded sample of the workload"},
        "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
        "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)



# ------------------------------------------------------------------------------- roofline
# What limits each kernel (profiles/r02_*_ncu_full.md): the whole-V-stage kernels are bound by instruction
# issue / latency (their DRAM rate is about half the copy rate at 100 % of the bytes they must move), every
# other kernel by HBM.
KERNEL_BOUND = {"fused_vx_vy_vz_moments": "issue", "fused_vx_vy_vz": "issue", "match_moments": "issue"}
COUNTERS = ROOT / "profiles" / "kernel_counters.json"


def csrc_sha16() -> str:
    """Hash of the CUDA sources: ncu counters in profiles/kernel_counters.json are only quoted while it matches."""
    import hashlib
    h = hashlib.sha256()
    for p in sorted((ROOT / "paper_2305_01487_b200" / "csrc").glob("*.cu*")):
        h.update(p.name.encode()); h.update(p.read_bytes())
    return h.hexdigest()[:16]


def sim_sm_count(torch, index: int) -> int:
    return int(torch.cuda.get_device_properties(index).multi_processor_count)


def make_roofline(timings, steps, ms_per_step, peak_gbs, peak_src, clocks, sm_count, w):
    """The roofline object of the bench line. For the dominant kernel (largest share of the step):
    achieved = bytes the launch MUST move (f read once + written once per pass, whatever it fuses) / its mean
    CUDA-event duration; frac = achieved / measured copy rate -- a physical fraction, <= ~1. The survey's
    contract currency (algorithmic bytes of the UNFUSED sweeps) is kept under *_algorithmic_unfused: fusion makes
    it exceed 1. traffic = DRAM bytes ncu measured for that kernel, quoted only while the sources are unchanged."""
    kern = {k: dict(v, ms_per_launch=v["ms"] / v["launches"]) for k, v in timings.items()}
    dom = max(kern, key=lambda k: kern[k]["ms"])
    d = kern[dom]
    total_ms = sum(v["ms"] for v in kern.values())
    step_alg = sum(v["alg_bytes"] * v["launches"] for v in kern.values()) / steps
    step_moved = sum(v["moved_bytes"] * v["launches"] for v in kern.values()) / steps
    achieved = d["moved_bytes"] / (d["ms_per_launch"] * 1e-3) / 1e9
    counters, note = {}, None
    try:
        cj = json.loads(COUNTERS.read_text())
        if cj.get("csrc_sha16") == csrc_sha16() and cj.get("workload") == w.name:
            counters = cj.get("kernels", {})
        else:
            note = (f"profiles/kernel_counters.json was measured at commit {cj.get('commit')} on {cj.get('workload')}; "
                    "the CUDA sources or the workload differ now, so no ncu counter is quoted")
    except Exception as e:  # noqa: BLE001
        note = f"no profiles/kernel_counters.json ({e!r})"
    cd = counters.get(dom, {})
    sm_hz = 1e6 * float(clocks.get("sm_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    issue_peak = sm_count * 4 * sm_hz                     # one warp instruction per scheduler per cycle
    r = {
        "bound": KERNEL_BOUND.get(dom, "hbm"), "kernel": dom,
        "achieved": achieved, "peak": peak_gbs, "unit": "GB/s", "frac": achieved / peak_gbs,
        "what": "bytes the dominant kernel must move per launch (one read + one write of f) / its CUDA-event time, "
                "against the measured copy rate",
        "peak_source": f"{peak_src} (MEASURED_PEAKS.json hbm_gbs)" if peak_src == "measured" else "fallback 6650 GB/s",
        "traffic": cd.get("dram_bytes"),
        "share_of_step": d["ms"] / total_ms,
        "frac_algorithmic_unfused": d["alg_bytes"] / (d["ms_per_launch"] * 1e-3) / 1e9 / peak_gbs,
        "step": {"moved_GBps": step_moved / (ms_per_step * 1e-3) / 1e9,
                 "frac": step_moved / (ms_per_step * 1e-3) / 1e9 / peak_gbs,
                 "algorithmic_unfused_GBps": step_alg / (ms_per_step * 1e-3) / 1e9,
                 "frac_algorithmic_unfused_of_8TBps": step_alg / (ms_per_step * 1e-3) / 8e12,
                 "frac_algorithmic_unfused_of_measured": step_alg / (ms_per_step * 1e-3) / 1e9 / peak_gbs},
        "kernels": {},
    }
    if note:
        r["traffic_note"] = note
    elif counters:
        r["traffic_source"] = f"profiles/kernel_counters.json (ncu --set full, commit {cj.get('commit')})"
    for k, v in kern.items():
        e = {"bound": KERNEL_BOUND.get(k, "hbm"), "ms_per_launch": round(v["ms_per_launch"], 4),
             "launches_per_step": v["launches"] / steps,
             "moved_GBps": round(v["moved_bytes"] / (v["ms_per_launch"] * 1e-3) / 1e9, 1),
             "frac": round(v["moved_bytes"] / (v["ms_per_launch"] * 1e-3) / 1e9 / peak_gbs, 4),
             "algorithmic_unfused_GBps": round(v["alg_bytes"] / (v["ms_per_launch"] * 1e-3) / 1e9, 1)}
        ck = counters.get(k, {})
        if ck.get("warp_instructions"):
            # issue roofline: executed warp instructions (ncu smsp__inst_executed.sum) / time against one
            # instruction per scheduler per cycle at the SM clock seen during the run
            rate = ck["warp_instructions"] / (v["ms_per_launch"] * 1e-3)
            e["issue"] = {"warp_instructions": ck["warp_instructions"],
                          "thread_instructions_per_cell": round(32.0 * ck["warp_instructions"] / w.n_cells, 2),
                          "achieved_Ginstr_s": round(rate / 1e9, 1), "peak_Ginstr_s": round(issue_peak / 1e9, 1),
                          "frac": round(rate / issue_peak, 4)}
            if ck.get("fp64_pipe_warp_instructions"):
                # the tight bound of these kernels: DADD / DMUL / DSETP occupy the fp64 pipe of a scheduler for 2 cycles
                # per warp instruction, a DFMA whose three operands are live registers (all of them here) for 3
                # (measured with a microbenchmark in round 2: profiles/r02_issue_rate.md)
                n64, nfma = ck["fp64_pipe_warp_instructions"], ck.get("dfma_warp_instructions", 0)
                cycles = 2.0 * (n64 - nfma) + 3.0 * nfma                 # pipe cycles summed over all schedulers
                floor_ms = cycles / (sm_count * 4) / sm_hz * 1e3
                e["fp64_pipe"] = {"warp_instructions": n64, "dfma_warp_instructions": nfma,
                                  "thread_instructions_per_cell": round(32.0 * n64 / w.n_cells, 2),
                                  "pipe_floor_ms": round(floor_ms, 4), "frac": round(floor_ms / v["ms_per_launch"], 4)}
        r["kernels"][k] = e
    for key in ("issue", "fp64_pipe"):
        if key in r["kernels"][dom]:
            r[key] = r["kernels"][dom][key]
    return r


# ------------------------------------------------------------------------------- CUDA arm
def run_mphv(args, w):
    import torch
    import torch.distributed as dist
    from paper_2305_01487_b200 import inputs, mphv

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl mphv needs a B200: there is no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        # NCCL's communicator log (ranks, transports, NVLS) on stderr, so that a run record shows the N ranks
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        dist.init_process_group("nccl", device_id=dev)
    halo_mode = args.decomp == "halo" or (args.decomp == "auto" and world > 1)
    if halo_mode:
        # one problem, N blocks along the periodic x axis (box and grid N times longer in x)
        from paper_2305_01487_b200 import halo
        wg = inputs.variant(w, name=f"{w.name}_x{world}", nx=(w.nx[0] * world, w.nx[1], w.nx[2]),
                            xhi=(w.xlo[0] + (w.xhi[0] - w.xlo[0]) * world, w.xhi[1], w.xhi[2]))
        dims = halo.choose_dims(wg.nx, world) if world > 1 else (1, 1, 1)    # x only: the fused X stage (mphv_stage_x_halo)
        assert dims == (world, 1, 1), dims
        dec = halo.Decomp(wg.nx, wg.bc, dims)
        Eg, Bg = inputs.make_fields(wg)
        dt = inputs.cfl_dt(wg, Eg, Bg)                       # same on every rank (global fields)
        sl = dec.local_slices(rank)
        E, B = (np.ascontiguousarray(a[(slice(None),) + sl]) for a in (Eg, Bg))
        wr = inputs.variant(dec.local_workload(wg, rank), seed_offset=1000 * rank)
        f0 = inputs.make_f0(wr)
    else:
        # each rank: its own seeded copy of the workload (independent problems => weak scaling)
        wr = inputs.variant(w, seed_offset=1000 * rank)
        f0, E, B, dt = inputs.make_all(wr)
    peaks = {}
    try:
        peaks = json.loads((ROOT / "MEASURED_PEAKS.json").read_text())
    except Exception:  # noqa: BLE001
        pass
    peak_gbs, peak_src = (float(peaks["hbm_gbs"]), "measured") if "hbm_gbs" in peaks else (6650.0, "fallback")

    if halo_mode:
        dv = halo.DistributedVlasov(wg, dec, rank, dev, force_halo=(0,) if world == 1 else False)
        sim = dv.sim
        step_moments = dv.step_moments
    else:
        sim = mphv.Vlasov.from_workload(wr, device=dev)
        step_moments = sim.step_moments
    sim.set_fusion(args.fusion)
    if args.vmode == "backsub":
        sim.set_vmode(mphv.V_BACKSUB)
    f = torch.from_numpy(f0).to(dev)
    sim.bind_f(f)
    sim.set_fields(torch.from_numpy(E).to(dev), torch.from_numpy(B).to(dev))
    mom = sim.alloc_moments()
    f_ref0 = f.clone() if w.n_cells <= 2 ** 28 else None

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(3, args.warmup)):
        step_moments(dt, mom)
    barrier()
    launches0 = sim.launches
    sim.set_timing(True)          # per-launch CUDA events inside the timed region (conservative: they cost a little)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    with ClockSampler(local) as clk:
        barrier()
        ev[0].record()
        for k in range(args.steps):
            step_moments(dt, mom)
            ev[k + 1].record()
        barrier()
    e0, e1 = ev[0], ev[-1]
    ms = e0.elapsed_time(e1)                                      # EXACTLY args.steps steps, one bracket
    per_step = sorted(ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps))   # the same steps, one by one
    launches = sim.launches - launches0
    timings = sim.timings()
    sim.set_timing(False)
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    ms_per_step = ms / args.steps
    value = w.n_cells * world * args.steps / (ms * 1e-3)

    # sanity of the timed state: f finite, non-negative, moments finite
    assert bool(torch.isfinite(mom[0]).all()) and float(f.min()) >= 0.0

    clocks = clk.summary()
    roofline = make_roofline(timings, args.steps, ms_per_step, peak_gbs, peak_src, clocks, sim_sm_count(torch, local), w)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(3, args.warmup), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "cells_per_gpu": w.n_cells, "bytes_per_copy_of_f": w.n_cells * 8,
                   "step": "S_x,S_y[,S_z],V_vx,V_vy,V_vz + moments n,j,P every step",
                   "l2": "inputs larger than L2 (f is %.2f GB >> 126 MB); no flush needed" % (w.n_cells * 8 / 1e9),
                   "fusion": args.fusion, "vmode": args.vmode,
                   "parallelism": "1 GPU" if world == 1 else
                   (f"{world} spatial blocks along periodic x, 2-layer halo exchange before S_x (NCCL send/recv), "
                    f"{2 * sim.halo_count(0) * 8} B sent per rank per step" if halo_mode else f"{world} independent problems")},
        "clocks": clocks, "gpu_launches": launches, "roofline": roofline,
        "ms_per_step_median": per_step[len(per_step) // 2], "ms_per_step_min": per_step[0], "ms_per_step_max": per_step[-1],
        "timing": f"one CUDA-event bracket around the {args.steps} steps (value, ms_per_step); median/min/max over the same "
                  f"{args.steps} steps timed one by one; per-launch CUDA events are recorded inside the timed region",
    }

    # end to end through the C ABI with HOST buffers: H2D(f) + step + moments + D2H(f, moments) per step
    if not args.no_e2e:
        fh = torch.from_numpy(f0).pin_memory()
        nh = torch.empty(wr.space_shape, dtype=torch.float64).pin_memory()
        jh = torch.empty((3,) + wr.space_shape, dtype=torch.float64).pin_memory()
        Ph = torch.empty((6,) + wr.space_shape, dtype=torch.float64).pin_memory()
        if halo_mode:
            def run_host_step():                                # the same traffic as mphv_run_host, with the exchange
                f.copy_(fh, non_blocking=True)
                step_moments(dt, mom)
                fh.copy_(f, non_blocking=True)
                nh.copy_(mom[0], non_blocking=True); jh.copy_(mom[1], non_blocking=True); Ph.copy_(mom[2], non_blocking=True)
                torch.cuda.synchronize()
        else:
            def run_host_step():
                sim.run_host(fh, 1, dt, nh, jh, Ph)
        run_host_step()                                         # warm-up
        barrier()
        t0 = time.perf_counter()
        e0.record()
        for _ in range(args.e2e_steps):
            run_host_step()
        e1.record()
        barrier()
        wall = time.perf_counter() - t0
        ems = max(e0.elapsed_time(e1), wall * 1e3)
        if world > 1:
            t = torch.tensor([ems], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ems = float(t.item())
        line["e2e"] = {"value": w.n_cells * world * args.e2e_steps / (ems * 1e-3), "unit": UNIT,
                       "h2d_bytes_per_step": w.n_cells * 8, "d2h_bytes_per_step": w.n_cells * 8 + 10 * wr.n_space * 8,
                       "ms_per_step": ems / args.e2e_steps, "steps": args.e2e_steps,
                       "what": ("pinned host f -> device, decomposed split step with halo exchange, moments, f and moments -> host"
                                if halo_mode else
                                "mphv_run_host: pinned host f -> device, full split step, moments, f and moments -> host; the library cuts f "
                                "into slabs along y and overlaps copy in, sweeps and copy out slab by slab")}
        del fh
        if not halo_mode:
            # coupled run, f resident: per step the host hands over E, B and gets n, j, P back
            Eh, Bh = torch.from_numpy(E).pin_memory(), torch.from_numpy(B).pin_memory()
            sim.step_fields_host(Eh, Bh, dt, nh, jh, Ph)            # warm-up
            barrier()
            t0 = time.perf_counter()
            for _ in range(args.steps):
                sim.step_fields_host(Eh, Bh, dt, nh, jh, Ph)
            barrier()
            wall = time.perf_counter() - t0
            if world > 1:
                t = torch.tensor([wall], dtype=torch.float64, device=dev)
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
                wall = float(t.item())
            line["e2e_resident"] = {"value": w.n_cells * world * args.steps / wall, "unit": UNIT,
                                    "h2d_bytes_per_step": 6 * wr.n_space * 8, "d2h_bytes_per_step": 10 * wr.n_space * 8,
                                    "ms_per_step": 1e3 * wall / args.steps, "steps": args.steps,
                                    "what": "mphv_step_fields_host: f stays on the device; pinned host E, B -> device, "
                                            "set_fields, full split step, moments -> host, stream sync every step (wall clock)"}

    if world == 1 and not halo_mode and not args.no_two_species and w.kind != "landau1d" and args.vmode == "plain":
        line["two_species"] = run_two_species(args, torch, mphv, inputs, w, sim, f, dev)

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        del f0
        line["cpu_baseline"] = {k: v for k, v in time_oracle(w, min(SAMPLE_STEPS, max(1, args.steps)), 1, args.cpu_seconds).items() if k != "ms_per_step"}

    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_two_species(args, torch, mphv, inputs, w, ions, f_ions, dev):
    """the paper's Scheme {Vlasov e, Vlasov i, Maxwell} on the workload's spatial grid.
    Ions = the workload (f as the timed run left it), electrons = inputs.electrons_of (q/m = -100, 36^3 on +-20,
    P:L215), FDTD Maxwell with c = 20; mphv_plasma_step (coupled step R22: per step 2 launches per species + 1
    field launch, no host sync). Timed serially (everything on one stream) and with one stream per species; the
    ratio says whether the SMs co-schedule one species' HBM-bound spatial sweeps with the other's issue-bound
    V stage. dt = half the CFL bound over both species' sweeps."""
    we = inputs.electrons_of(w)
    fe = torch.from_numpy(inputs.make_f0(we)).to(dev)
    Ey, By = inputs.yee_fields(w)
    dt = 0.5 * min(inputs.cfl_dt(w, 2 * Ey, 2 * By), inputs.cfl_dt(we, 2 * Ey, 2 * By))
    el = mphv.Vlasov.from_workload(we, device=dev)
    el.bind_f(fe)
    mx = mphv.Maxwell.from_workload(w, c2=400.0, inv_eps0=1.0, device=dev)
    Ed, Bd = torch.from_numpy(Ey).to(dev), torch.from_numpy(By).to(dev)
    mx.bind(Ed, Bd)
    pl = mphv.Plasma(mx, [ions, el], [1.0, -1.0])
    cells = w.n_cells + we.n_cells
    steps = max(2, args.species_steps)
    out = {"what": "mphv_plasma_step: ions (the workload) + electrons (%s, q/m = -100) + FDTD Maxwell, coupled step R22; "
                   "value = cells of both species x steps / time (CUDA events on the field stream, which joins the species' streams)" % we.name,
           "cells": {"ions": w.n_cells, "electrons": we.n_cells}, "steps": steps, "unit": UNIT}
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for mode in ("serial", "concurrent"):
        pl.set_concurrent(mode == "concurrent")
        pl.step(dt, 2)
        pl.sync()
        l0 = ions.launches + el.launches
        e0.record()
        pl.step(dt, steps)
        e1.record()
        pl.sync()
        ms = e0.elapsed_time(e1)
        out[mode] = {"ms_per_step": ms / steps, "value": cells * steps / (ms * 1e-3),
                     "species_launches_per_step": (ions.launches + el.launches - l0) / steps}
    out["speedup_concurrent_over_serial"] = out["serial"]["ms_per_step"] / out["concurrent"]["ms_per_step"]
    n_i = pl.moments(0)[0]
    assert bool(torch.isfinite(n_i).all()) and bool(torch.isfinite(Ed).all()) and float(fe.min()) >= 0.0
    pl.close()
    return out


def run_aux(args, w):
    """Device times (CUDA events in the library, per launch) of mphv_maxwellian, mphv_exchange_maxwellian and
    mphv_match_moments on workload w; algorithmic bytes: 8 per cell written (fill), 16 per boundary cell
    (exchange: f_ext read, ghost written), 24 per cell (matching: f read for its moments, read again, written)."""
    import torch
    from paper_2305_01487_b200 import inputs, mphv
    dev = torch.device("cuda", 0)
    f0, E, B, dt = inputs.make_all(w)
    sim = mphv.Vlasov.from_workload(w, device=dev)
    f = torch.from_numpy(f0).to(dev)
    sim.bind_f(f)
    sim.set_fields(torch.from_numpy(E).to(dev), torch.from_numpy(B).to(dev))
    n, j, P = sim.step_moments(dt)
    ns = w.n_space
    n1, j1, P1 = n.reshape(-1).contiguous(), j.reshape(3, -1).contiguous(), P.reshape(6, -1).contiguous()
    out = torch.empty_like(f)
    dim = 1 if w.nx[1] >= 4 else 0
    plane = ns // w.nx[dim]
    nf = torch.ones(2 * plane, dtype=torch.float64, device=dev)
    jf = torch.zeros(6 * plane, dtype=torch.float64, device=dev)
    Pf = torch.zeros(6, 2 * plane, dtype=torch.float64, device=dev)
    Pf[0] = Pf[3] = Pf[5] = 1.0
    for rep in range(2):                                  # first pass = warm-up
        sim.set_timing(True)
        for _ in range(args.steps):
            sim.maxwellian(n1, j1, P1, out=out.view(ns, w.nv[2], w.nv[1], w.nv[0]))
            sim.exchange_maxwellian(dim, 1, nf, jf, Pf)
            sim.match_moments(n, j, P)
        torch.cuda.synchronize()
        t = sim.timings()
        sim.set_timing(False)
    kern = {k: {"ms_per_launch": round(v["ms"] / v["launches"], 4),
                "alg_GBps": round(v["alg_bytes"] / (v["ms"] / v["launches"] * 1e-3) / 1e9, 1)} for k, v in t.items()}
    print(json.dumps({"metric": "aux_kernels", "config": {"workload": w.name, "cells": w.n_cells,
                      "exchange": f"axis {dim}, high end, {2 * plane} boundary cells"},
                      "dtype": "f64", "data": "synthetic", "kernels": kern}), flush=True)


def main():
    args = parse()
    from paper_2305_01487_b200 import inputs
    w = inputs.config(args.config)
    if args.aux:
        run_aux(args, w)
    elif args.impl == "reference":
        run_reference(args, w)
    else:
        run_mphv(args, w)


if __name__ == "__main__":
    main()
