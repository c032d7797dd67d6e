#!/usr/bin/env python
"""bench.py -- TDGL cell-updates/s of the hand-written sm_100a hot path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5a|cfg5b|cfg3|cfg1] [--dtype f64|f32]
    python bench.py --impl reference ...      # the CPU oracle on a bounded sample (rank 0 only)

A step = one forward-Euler step of the whole hot path (pruned x/y transforms, fused z
transform + tensor multiply, inverse transforms, fused local step) over the synthetic workload.  One JSON line
is printed by rank 0.  N > 1: every rank runs an independent replica of the workload (batch sharding, no
data-path collective), value = all ranks' cell-updates / max-over-ranks time.  Started
without a torchrun environment, `--gpus N` (N > 1) re-executes itself under torch.distributed.run with N ranks.
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
sys.path.insert(0, ROOT)

import fe_inputs as fi  # noqa: E402

METRIC = "TDGL cell-updates/s (fp64, incl. FFT electrostatics)"
UNIT = "cell-updates/s"


def make_workload(name: str, dtype: str) -> fi.Workload:
    if name == "cfg5a":
        return fi.config5a(dtype)
    if name == "cfg5b":
        return fi.config5b(dtype)
    if name == "cfg3":
        w = fi.config3()
        w.dtype = dtype
        return w
    if name == "cfg1":
        w = fi.config1()
        w.dtype = dtype
        return w
    raise SystemExit("unknown workload " + name)


def sample_workload(name: str) -> fi.Workload:
    """Bounded sample of the benchmark workload for the CPU oracle: one member of config 5b
    (128x128x64 cells, the same recipe as 5a: BaTiO3 300 K, 1 nm cells, open boundaries, |P| = 0.26 sphere-uniform,
    Euler dt* = 0.002) instead of the 256x256x128 cells of config 5a."""
    if name == "cfg1":
        return fi.config1()
    return fi.open_batio3("cfg5b_member0_128x128x64", (128, 128, 64), 1, "f64", 1005)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            return json.load(fh), "measured"
    return {"hbm_gbs": 6650.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
            # the first query initialises NVML and can stall the GPU for tens of ms: wait for it outside the timed region
            t_end = time.time() + 3.0
            while not self.rows and time.time() < t_end:
                time.sleep(0.02)
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.25)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------------
def padded_dims(w: fi.Workload):
    """Transform length per axis: the axis itself when periodic, the power of two >= 2 n when open (A16)."""
    m = []
    for a in range(3):
        if w.periodic[a]:
            m.append(w.n[a])
        else:
            v = 4
            while v < 2 * w.n[a]:
                v *= 2
            m.append(v)
    return m


def moved_bytes(w: fi.Workload, rsz: int):
    """Bytes each kernel of the CURRENT pipeline must read and write once per launch: spectra
    counted with Lx = m_x/2 + 1 columns, E_elec materialised between the x inverse pass and the local step."""
    nx, ny, nz = w.n
    m = padded_dims(w)
    Lx, B, c = m[0] // 2 + 1, w.batch, 2 * rsz
    N = nx * ny * nz
    return {
        "xfwd": B * 3 * (N * rsz + nz * ny * Lx * c),
        "yfwd": B * 3 * (nz * ny * Lx * c + nz * m[1] * Lx * c),
        "zmul": B * 3 * 2 * nz * m[1] * Lx * c + 6 * (m[2] // 2 + 1) * (m[1] // 2 + 1) * Lx * rsz,
        "yinv": B * 3 * (nz * ny * Lx * c + nz * m[1] * Lx * c),
        "xinv": B * 3 * (N * rsz + nz * ny * Lx * c),
        "local": B * 3 * N * rsz * 3,          # read P, read E_elec, write P_new
        # fused x + y passes: the half spectrum S1 stays in L2 (ring of planes), only P in and S2 out touch HBM
        "xyfwd": B * 3 * (N * rsz + nz * m[1] * Lx * c),
        "xyinv": B * 3 * (N * rsz + nz * m[1] * Lx * c),
    }


def survey_bytes_per_cell(w: fi.Workload, rsz: int) -> float:
    """SURVEY.md 8(d) "Algorithmic bytes per cell-RHS": per component s (1 + 4 p_x + 4 p_x p_y) with p_a = m_a / n_a,
    tensor 6 s p_x p_y p_z / 8 shared by the B members, local step 3 s read + 3 s write (E_elec consumed on chip):
    696 B for the open fp64 case at B = 1 (660 at B = 4, 651 at B = 16), 348 B in fp32."""
    m = padded_dims(w)
    px, py, pz = (m[a] / w.n[a] for a in range(3))
    return 3 * rsz * (1 + 4 * px + 4 * px * py) + 6 * rsz * px * py * pz / 8 / w.batch + 6 * rsz


_peaks_lib = None


def peaks_lib():
    """libfe_peaks.so: bench.py's own harness kernels (csrc/bench_peaks.cu); not part of the product library."""
    global _peaks_lib
    if _peaks_lib is None:
        import ctypes
        from paper_2605_28800_b200 import build as b
        L = ctypes.CDLL(b.PEAKS_LIB)
        vp, dp = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double)
        L.fe_peak_fp64.argtypes = [vp, ctypes.c_int, ctypes.c_int, dp, vp]
        L.fe_peak_lds.argtypes = [vp, ctypes.c_int, ctypes.c_int, dp, vp]
        L.fe_peak_l2.argtypes = [vp, vp, ctypes.c_int64, ctypes.c_int, dp, vp]
        L.fe_bench_kmul.argtypes = [vp, vp, vp, ctypes.c_int64, ctypes.c_int, ctypes.c_int, vp]
        _peaks_lib = L
    return _peaks_lib


def measure_unit_peaks(torch, dev):
    """fp64 issue rate, shared-memory and L2 read bandwidth of THIS box, timed with CUDA events inside the harness
    library (SURVEY.md 8(d) "Which roofline": the ALU bound is reported beside the HBM bound)."""
    import ctypes
    L = peaks_lib()
    st = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    scratch = torch.zeros(148 * 8 * 256 * 4, dtype=torch.float64, device=dev)
    out = ctypes.c_double(0.0)
    res = {}
    if L.fe_peak_fp64(ctypes.c_void_p(scratch.data_ptr()), 4, 4096, ctypes.byref(out), st) == 0:
        res["fp64_warp_inst_per_s"] = out.value
        res["fp64_tflops"] = out.value * 64 / 1e12          # one DFMA warp instruction = 32 lanes x 2 flops
    if L.fe_peak_lds(ctypes.c_void_p(scratch.data_ptr()), 4, 4096, ctypes.byref(out), st) == 0:
        res["lds_gbs"] = out.value / 1e9
    buf = torch.zeros(32 * 1024 * 1024 // 8, dtype=torch.float64, device=dev)       # 32 MB: fits L2
    if L.fe_peak_l2(ctypes.c_void_p(buf.data_ptr()), ctypes.c_void_p(scratch.data_ptr()), buf.numel() * 8, 20,
                    ctypes.byref(out), st) == 0:
        res["l2_read_gbs"] = out.value / 1e9
    return res


def ncu_counters(workload: str, dtype: str):
    """Per-launch counters of the committed ncu capture (profiles/ncu_traffic.json): DRAM bytes, fp64-pipe warp
    instructions and shared-memory wavefronts per kernel."""
    tp = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if not os.path.exists(tp):
        return {}
    with open(tp) as fh:
        return json.load(fh).get("%s_%s" % (workload, dtype), {})


def run_cuda(args):
    import torch
    import torch.distributed as dist
    import paper_2605_28800_b200 as fe
    from paper_2605_28800_b200 import parallel as par

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
    fe.load()

    w = make_workload(args.workload, args.dtype)
    rsz = 8 if args.dtype == "f64" else 4
    g = fe.Grid.from_workload(w, device=dev, dtype=args.dtype)
    g.set_option(fe.FE_OPT_FUSE_XY, args.fuse_xy)
    if args.xy_ring:
        g.set_option(fe.FE_OPT_XY_RING, args.xy_ring)
    g.set_option(fe.FE_OPT_XL_SLABS, args.xl_slabs)
    t0 = time.time()
    g.precompute_tensor()
    t_pre = time.time() - t0
    P_host = torch.from_numpy(w.P0.astype(np.float64 if args.dtype == "f64" else np.float32)).pin_memory()
    P = P_host.to(dev, non_blocking=False).contiguous()
    cells = w.cells * w.batch

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: W warm-up steps, then exactly K steps in one fe_step call -------------
    # warm-up: the W requested steps, then more until the GPU has been busy for ~0.5 s (a cold device ramps its clocks
    # and power state over the first tenths of a second: the first run on a fresh box was 10 % slow without this).
    # The JSON line prints both the requested and the executed count.
    g.step(P, w.dt, args.warmup, fe.FE_EULER, fe.FE_TERM_ALL)
    torch.cuda.synchronize()
    warm, t_w = args.warmup, time.perf_counter()
    while time.perf_counter() - t_w < 0.5 and warm < args.warmup + 2000:
        g.step(P, w.dt, 20, fe.FE_EULER, fe.FE_TERM_ALL)
        torch.cuda.synchronize()
        warm += 20
    P.copy_(P_host)                       # the timed steps start from the workload's initial state
    barrier()
    l0 = g.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as cs:
        torch.cuda.synchronize()
        ev0.record()
        g.step(P, w.dt, args.steps, fe.FE_EULER, fe.FE_TERM_ALL)
        ev1.record()
        barrier()
    launches = g.launch_count() - l0
    # whole-job throughput: all ranks' cell-updates / the slowest rank's device time
    value, ms = par.throughput(ev0.elapsed_time(ev1), float(cells * args.steps), device=dev)
    en = g.energy(P)[0]

    # ---- per-kernel durations, measured live with CUDA events on the launching stream (second pass of K steps)
    g.profile(True)
    g.step(P, w.dt, args.steps, fe.FE_EULER, fe.FE_TERM_ALL)
    prof = g.profile_read()
    g.profile(False)
    alg = moved_bytes(w, rsz)
    alg = {k: v for k, v in alg.items() if prof.get(k, (0, 0))[1]}          # the kernels that actually ran
    pk, pk_kind = peaks()
    hbm = pk["hbm_gbs"]
    unit = measure_unit_peaks(torch, dev) if rank == 0 else {}
    ctr = ncu_counters(args.workload, args.dtype)
    kern = {}
    for k, (tms, cnt) in prof.items():
        if cnt and k in alg:
            dur = tms / cnt
            row = {"ms": dur, "alg_gbs": alg[k] / (dur * 1e-3) / 1e9, "frac_hbm": alg[k] / (dur * 1e-3) / 1e9 / hbm,
                   "launches": cnt}
            c = ctr.get(k) if isinstance(ctr.get(k), dict) else None
            if c and unit.get("fp64_warp_inst_per_s") and c.get("fp64_warp_inst"):
                row["frac_fp64"] = c["fp64_warp_inst"] / (dur * 1e-3) / unit["fp64_warp_inst_per_s"]
            if c and unit.get("lds_gbs") and c.get("smem_wavefronts"):
                row["frac_lds"] = c["smem_wavefronts"] * 128 / (dur * 1e-3) / 1e9 / unit["lds_gbs"]
            kern[k] = row
    prof_total = sum(v["ms"] for v in kern.values())
    dom = max(kern, key=lambda k: kern[k]["ms"])
    cdom = ctr.get(dom) if isinstance(ctr.get(dom), dict) else {}
    traffic = cdom.get("dram_bytes") if cdom else (ctr.get(dom) if not isinstance(ctr.get(dom), dict) else None)
    # kernel that serves the profile slot on the size-specialised path (every bench workload but cfg1 takes it)
    # barrier-free x kernels: padded half length 256 (fp64, fp32) or 128 / 64 (fp64) on an open x axis
    mxh = padded_dims(w)[0] // 2
    k6 = (not w.periodic[0]) and (mxh == 256 or (args.dtype == "f64" and mxh in (64, 128)))
    fast_names = {"xfwd": "k6_xfwd" if k6 else "k2_xfwd", "yfwd": "k4_axis<-1>", "zmul": "k2_zmul", "yinv": "k4_axis<+1>",
                  "xinv": "k6_xinv" if k6 else "k2_xinv",
                  "local": "k_local2", "xyfwd": "k_xyfwd", "xyinv": "k_xyinv"}
    generic = args.workload == "cfg1"
    # which roofline binds the dominant kernel: the largest of its fractions of the three measured unit peaks
    fr = {"hbm": kern[dom]["frac_hbm"], "alu": kern[dom].get("frac_fp64", 0.0), "lds": kern[dom].get("frac_lds", 0.0)}
    bound = max(fr, key=lambda k: fr[k])
    step_s = ms / args.steps * 1e-3
    sv = survey_bytes_per_cell(w, rsz)
    roofline = {"bound": bound, "bound_fracs": fr,
                "kernel": ("k_" + dom) if generic else fast_names.get(dom, "k_" + dom),
                "achieved": kern[dom]["alg_gbs"], "peak": hbm,
                "peak_kind": pk_kind + " (burst copy bandwidth, MEASURED_PEAKS.json)", "unit": "GB/s",
                "frac": kern[dom]["alg_gbs"] / hbm, "traffic": traffic,
                "share_of_step": kern[dom]["ms"] / prof_total,
                "alu": None, "lds": None,
                "whole_step": {"alg_bytes_per_cell": sv, "alg_model": "SURVEY.md 8(d): E_elec on chip, m_x/2 columns",
                               "moved_bytes_per_cell": sum(alg.values()) / cells,
                               "achieved": sv * cells / step_s / 1e9,
                               "frac": sv * cells / step_s / 1e9 / hbm,
                               "frac_of_nominal_8000": sv * cells / step_s / 1e9 / 8000.0,
                               "moved_frac": sum(alg.values()) / step_s / 1e9 / hbm},
                "unit_peaks": unit, "kernels": kern}
    if unit.get("fp64_warp_inst_per_s") and cdom.get("fp64_warp_inst"):
        ach = cdom["fp64_warp_inst"] / (kern[dom]["ms"] * 1e-3)
        roofline["alu"] = {"peak": unit["fp64_warp_inst_per_s"], "peak_kind": "measured (dependent DFMA chains, bench_peaks.cu)",
                           "unit": "fp64 warp-inst/s", "achieved": ach, "frac": ach / unit["fp64_warp_inst_per_s"],
                           "inst_per_launch": cdom["fp64_warp_inst"], "inst_source": "ncu sm__inst_executed_pipe_fp64 (profiles/ncu_traffic.json)"}
    if unit.get("lds_gbs") and cdom.get("smem_wavefronts"):
        ach = cdom["smem_wavefronts"] * 128 / (kern[dom]["ms"] * 1e-3) / 1e9
        roofline["lds"] = {"peak": unit["lds_gbs"], "peak_kind": "measured (conflict-free 128-bit LDS, bench_peaks.cu)",
                           "unit": "GB/s", "achieved": ach, "frac": ach / unit["lds_gbs"],
                           "wavefronts_per_launch": cdom["smem_wavefronts"]}

    # ---- end to end through the C ABI with host buffers: every step copies its input state from pinned host memory,
    # runs one step and copies the result back to pinned host memory.  Serial: the three phases back to back.
    # Pipelined (the reported value): a ring of three device buffers, H2D / step / D2H on three streams, so the upload of
    # job i+1 and the download of job i-1 overlap the step of job i and the upload stream never waits for a download
    # (independent jobs, PCIe is full duplex).
    NB = 3
    out_host = [torch.empty(P_host.shape, dtype=P_host.dtype, pin_memory=True) for _ in range(NB)]
    nbytes = P_host.numel() * P_host.element_size()
    e2e_steps = max(2, min(args.steps, 32))
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        P.copy_(P_host, non_blocking=True)
        g.step(P, w.dt, 1, fe.FE_EULER, fe.FE_TERM_ALL)
        out_host[0].copy_(P, non_blocking=True)
        torch.cuda.synchronize()
    serial_value, _ = par.throughput((time.perf_counter() - t0) * 1e3, float(cells * e2e_steps), device=dev)
    bufs = [P] + [torch.empty_like(P) for _ in range(NB - 1)]
    s_in, s_out, s_cmp = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.current_stream()
    ev_in = [torch.cuda.Event() for _ in range(NB)]
    ev_done = [torch.cuda.Event() for _ in range(NB)]
    ev_out = [torch.cuda.Event() for _ in range(NB)]
    barrier()
    t0 = time.perf_counter()
    for i in range(e2e_steps):
        b = i % NB
        with torch.cuda.stream(s_in):
            if i >= NB:
                s_in.wait_event(ev_out[b])              # the previous result of this buffer has left the device
            bufs[b].copy_(P_host, non_blocking=True)
            ev_in[b].record(s_in)
        s_cmp.wait_event(ev_in[b])
        g.step(bufs[b], w.dt, 1, fe.FE_EULER, fe.FE_TERM_ALL)
        ev_done[b].record(s_cmp)
        with torch.cuda.stream(s_out):
            s_out.wait_event(ev_done[b])
            out_host[b].copy_(bufs[b], non_blocking=True)
            ev_out[b].record(s_out)
    torch.cuda.synchronize()
    e2e_value, _ = par.throughput((time.perf_counter() - t0) * 1e3, float(cells * e2e_steps), device=dev)
    e2e = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
           "steps": e2e_steps, "mode": "pinned host buffers; H2D, fe_step, D2H on three streams, ring of three device buffers",
           "serial_value": serial_value}
    del bufs

    # ---- cuFFT comparison (timed baseline, not the product): unpruned pad + rfftn + multiply + irfftn + crop
    cufft = None
    if rank == 0 and not args.no_cufft:
        try:
            cufft = cufft_pipeline_ms(torch, w, args.dtype, dev)
            ours = sum(kern[k]["ms"] for k in ("xfwd", "yfwd", "xyfwd", "zmul", "yinv", "xinv", "xyinv") if k in kern)
            cufft["ours_ms"] = ours
            cufft["speedup"] = cufft["ms_tight"] / ours
            cufft["speedup_vs_eager"] = cufft["ms_eager"] / ours
        except Exception as exc:      # out of memory on small boxes etc.: report, do not fail the bench
            cufft = {"error": str(exc)[:200]}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cpu = cpu_baseline(args.workload)

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": warm, "warmup_requested": args.warmup_requested,
                "warmup_note": "requested steps, then 20-step batches until the device has been busy for 0.5 s",
                "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
                "config": {"workload": w.name, "grid": list(w.n), "batch": w.batch, "integrator": "euler",
                           "terms": "landau+gradient+elec+ext", "padded_fft": padded_dims(w),
                           "l2": "state and spectra exceed L2 (P 3N reals, spectra >= 4x that)",
                           "parallelism": "replicas x%d" % world, "fuse_xy": args.fuse_xy, "xl_slabs": args.xl_slabs},
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches),
                "clocks": cs.summary(), "cufft_baseline": cufft, "precompute_s": t_pre,
                "energy_after": {"F_tot": float(en[4]), "finite": bool(np.isfinite(en).all())}}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def cufft_pipeline_ms(torch, w, dtype, dev):
    """The paper's design (cuFFT + custom kernels for the intermediate operations) on the same sizes:
    pad copy, rfftn of the padded box, 6-component multiply, irfftn, crop.  Timed twice: `tight` = padded box, spectrum
    and output preallocated, plans warm, the multiply one fused harness kernel (bench_peaks.cu: fe_bench_kmul), the crop a
    view; `eager` = the same written with eager tensor arithmetic and fresh allocations (round 1's figure)."""
    import ctypes
    td = torch.float64 if dtype == "f64" else torch.float32
    nx, ny, nz = w.n
    m = padded_dims(w)
    B = w.batch
    hx = m[0] // 2 + 1
    P = torch.randn(B, 3, nz, ny, nx, device=dev, dtype=td)
    K6 = torch.randn(6, m[2], m[1], hx, device=dev, dtype=td)
    idx = ((0, 3, 4), (3, 1, 5), (4, 5, 2))
    L = peaks_lib()
    st = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)

    Pp = torch.zeros(B, 3, m[2], m[1], m[0], device=dev, dtype=td)          # padding zeroed once: only the corner changes
    nk = m[2] * m[1] * hx

    def tight():
        Pp[:, :, :nz, :ny, :nx].copy_(P)
        Ph = torch.fft.rfftn(Pp, dim=(2, 3, 4))
        Eh = torch.empty_like(Ph)
        if L.fe_bench_kmul(ctypes.c_void_p(Ph.data_ptr()), ctypes.c_void_p(K6.data_ptr()), ctypes.c_void_p(Eh.data_ptr()),
                           nk, B, 0 if dtype == "f64" else 1, st) != 0:
            raise RuntimeError("fe_bench_kmul failed")
        del Ph
        return torch.fft.irfftn(Eh, s=(m[2], m[1], m[0]), dim=(2, 3, 4))[:, :, :nz, :ny, :nx]

    def eager():
        Pq = torch.zeros(B, 3, m[2], m[1], m[0], device=dev, dtype=td)
        Pq[:, :, :nz, :ny, :nx] = P
        Ph = torch.fft.rfftn(Pq, dim=(2, 3, 4))
        del Pq
        Eh = torch.stack([sum(K6[idx[i][j]] * Ph[:, j] for j in range(3)) for i in range(3)], dim=1)
        del Ph
        return torch.fft.irfftn(Eh, s=(m[2], m[1], m[0]), dim=(2, 3, 4))[:, :, :nz, :ny, :nx].contiguous()

    def timeit(fn, reps):
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    t_tight = timeit(tight, 5)
    t_eager = timeit(eager, 3)
    return {"ms": t_tight, "ms_tight": t_tight, "ms_eager": t_eager,
            "what": "torch.fft.rfftn/irfftn (cuFFT) on the padded box; tight = preallocated padded box (zeroed once), warm "
                    "plans, one fused multiply kernel, crop as a view; eager = fresh allocations and eager tensor arithmetic"}


# ---------------------------------------------------------------------------------------------------------
def oracle_steps(workload: str, steps: int, warmup: int, threads: int):
    """Time the CPU oracle as it stands (oracle-FFT electrostatics O8 + Landau + gradient + Euler) on the sample.
    threads = 1: numpy.fft and one OpenMP thread; threads > 1: scipy.fft workers and that many OpenMP threads."""
    os.environ["OMP_NUM_THREADS"] = str(threads)
    from oracle import fe_oracle as orc
    w = sample_workload(workload)
    p = orc.Problem(n=w.n, d=w.d, periodic=w.periodic, pbc_images=w.pbc_images, materials=w.materials[0],
                    g=w.globals_[0], matmap=w.matmap)
    o = orc.Oracle(p, elec="fft", fft_workers=threads if threads > 1 else None)
    o.table()                                  # tensor table: once per geometry, outside the timed region
    P = w.P0[0].copy()
    for _ in range(warmup):
        P = o.step(P, w.dt, 1, fi.EULER, fi.TERM_ALL)
    t0 = time.perf_counter()
    for _ in range(steps):
        P = o.step(P, w.dt, 1, fi.EULER, fi.TERM_ALL)
    dt = time.perf_counter() - t0
    oracle_steps.last = (o, P, w)
    return w, dt


def oracle_single_thread_step():
    """One more Euler step of the oracle object just timed, on ONE host thread (numpy.fft, one OpenMP thread): the
    single-thread figure beside the all-cores one.  Returns seconds, or None when the OpenMP runtime cannot be reached."""
    import ctypes
    o, P, w = oracle_steps.last
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(1)
    except OSError:
        return None
    o.fft_workers = None
    t0 = time.perf_counter()
    o.step(P, w.dt, 1, fi.EULER, fi.TERM_ALL)
    return time.perf_counter() - t0


def host_threads() -> int:
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:
        return max(1, os.cpu_count() or 1)


def cpu_baseline(workload: str):
    """the oracle on all host cores of the box (OpenMP loops + threaded library FFT), on one
    member of config 5b, 3 Euler steps after 1 warm-up step; tensor table outside the timed region."""
    th = host_threads()
    w, dt = oracle_steps(workload, 3, 1, th)
    dt1 = oracle_single_thread_step()
    return {"value": w.cells * 3 / dt, "unit": UNIT, "cores": th, "kind": "oracle",
            "single_thread_value": (w.cells / dt1) if dt1 else None,
            "sample": "%s: %dx%dx%d cells of the same recipe, 3 Euler steps, oracle-FFT electrostatics (scipy.fft, %d workers) "
                      "+ OpenMP C loops for Landau / gradient; tensor table built outside the timed region"
                      % (w.name, *w.n, th), "host_cores": os.cpu_count()}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    steps, warm = args.steps, min(args.warmup, 1)
    steps = min(steps, 10)
    th = host_threads()
    w, dt = oracle_steps(args.workload, steps, warm, th)
    value = w.cells * steps / dt
    sample = "%s (%dx%dx%d cells, same recipe as %s), %d Euler steps, %d host threads" % (w.name, *w.n, args.workload, steps, th)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
            "steps": steps, "warmup": warm, "ms_per_step": dt / steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": make_workload_name(args.workload), "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": th, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def make_workload_name(name: str) -> str:
    return {"cfg5a": "cfg5a_256x256x128", "cfg5b": "cfg5b_128x128x64_b4", "cfg3": "cfg3_sweep_64^3_b16",
            "cfg1": "cfg1_tiny_16x16x8"}[name]


def spawn_ranks(args) -> int:
    """`python bench.py --gpus N` outside torchrun: start N ranks (one per GPU) of this same script under
    torch.distributed.run, rendezvous on 127.0.0.1, and pass the exit code on."""
    import socket
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit("bench.py --gpus %d: only %d CUDA device(s) visible" % (args.gpus, have))
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="cfg5a", choices=["cfg5a", "cfg5b", "cfg3", "cfg1"])
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-cufft", action="store_true", help="skip the cuFFT comparison leg")
    ap.add_argument("--fuse-xy", type=int, default=0, choices=[0, 1],
                    help="FE_OPT_FUSE_XY: 1 = x and y passes fused through the L2 ring, 0 = separate kernels (default)")
    ap.add_argument("--xy-ring", type=int, default=0, help="FE_OPT_XY_RING (0 = automatic)")
    ap.add_argument("--xl-slabs", type=int, default=0,
                    help="FE_OPT_XL_SLABS: n > 1 = x inverse pass and local step slab by slab, E_elec handed over in L2")
    args = ap.parse_args()
    args.warmup_requested = args.warmup
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(args))
    else:
        if args.gpus != int(os.environ.get("WORLD_SIZE", "1")):
            raise SystemExit("bench.py: --gpus %d does not match WORLD_SIZE=%s" % (args.gpus, os.environ.get("WORLD_SIZE")))
        run_cuda(args)


if __name__ == "__main__":
    main()
