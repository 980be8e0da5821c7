#!/usr/bin/env python
"""bench.py -- throughput of the MMC hot path (cell updates/s) on synthetic meshes shaped like BASELINE.json's configs.

    python bench.py --gpus N --steps K --warmup W [--config 1..5] [--impl reference]

A "step" is one whole MMC iteration of the hot path: demag pack/pad -> forward FFT -> tensor multiply ->
inverse FFT + crop -> red colour pass -> black colour pass -> end-of-sweep bookkeeping (acceptance counters, running
means, cone controller).  `value` = (non-empty cells x steps) / device time, inputs resident in HBM; `e2e` = the same
through the C ABI with HOST buffers (pinned H2D of m before and D2H of m + observables after every step).
Multi-GPU: every rank runs an independent replica (own seed), no data-path collective;
value = total updates of all ranks / max-over-ranks device time.
`--impl reference` times the fp64 CPU oracle as it stands on the host cores on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "cell_updates_per_sec"
UNIT = "cell updates/s"
# Algorithmic (compulsory) bytes, DESIGN.md section 6.
# Colour pass, per cell update: own m read 12 + write 12, B_d 12 (demag configs), + 1 mask byte (open boundaries, empty
# cells) or + 4 (the class word = coefficient class << 7 | mask, cfg 4; SURVEY's alternative to 28 B of per-cell
# coefficients).  Units per launch = non-empty cells of one colour.
def layout_flags(wl):
    """(per-cell classes?, mask byte?, per-cell Ms0 array?) as libmmc_b200 decides them for this workload."""
    nonempty = [r for r in wl.regions if r["Ms0"] > 0]
    percell = wl.T_per_cell is not None or len(nonempty) > 1
    open_bc = any(n > 1 and not (wl.pbc_mask >> a) & 1 for a, n in enumerate((wl.nx, wl.ny, wl.nz)))
    mask = open_bc or wl.n_active < wl.N or (len(nonempty) > 1 and not wl.inter_region_exchange)
    ms0_per_cell = wl.n_active < wl.N or len({r["Ms0"] for r in nonempty}) > 1
    return percell, mask, ms0_per_cell


def pass_bytes_per_update(wl):
    percell, mask, _ = layout_flags(wl)
    return 24 + (12 if wl.demag else 0) + (4 if percell else (1 if mask else 0))


def _pow2_at_least(n, start):
    p = start
    while p < 2 * n - 1:
        p *= 2
    return p


def demag_layout(wl):
    """Which demag path libmmc_b200 takes for this mesh (mirrors demag_create): register-resident rows/columns kernels for
    padded lengths 2^8..2^12; with several layers a z-DFT of the shortest linear length 2 nz - 1 (fused into the columns kernel's
    loader) with a separate inverse z pass, or, with MMC_LP=1 and nz * Py/16 <= 512 threads, the layer-pair columns kernel."""
    Px, Py = _pow2_at_least(wl.nx, 2), _pow2_at_least(wl.ny, 1)
    fast = 8 <= (Px // 2).bit_length() - 1 <= 11 and 8 <= Py.bit_length() - 1 <= 12 and wl.nz <= 16
    lp = fast and wl.nz > 1 and (Py // 16) * wl.nz <= 512 and os.environ.get("MMC_LP", "0")[:1] == "1"   # an option; the z-DFT path is the default
    Pz = 1 if wl.nz == 1 else (2 * wl.nz - 1 if fast else _pow2_at_least(wl.nz, 1))
    return Px, Py, Pz, fast, lp


def demag_kernel_bytes(wl, ms0_per_cell):
    """Algorithmic bytes and flops per launch of the demag kernels (units per launch = the N mesh cells of one convolution).
    U = the layers' transposed half-spectra [3][nz][Px/2+1][ny] complex64 that the rows kernels write / read (only the ny kept
    rows are ever stored).  Layer-pair path: the columns kernel transforms U in place and reads the tensor spectra of the nz
    layer offsets: (4 + 6 (nz-1)) real arrays [Px/2+1][Py].  z-DFT path: the columns kernel reads U, writes the Pz planes
    T = [3][Pz][Px/2+1][ny] and reads 6 (4 for one layer) real arrays [Pz/2+1][Px/2+1][Py]; z_inverse reads T, writes U."""
    import math
    Px, Py, Pz, fast, lp = demag_layout(wl)
    Cx = Px // 2 + 1
    U = 3 * wl.nz * Cx * wl.ny * 8
    state = 3 * wl.N * 4
    fl_rows = 3 * wl.ny * wl.nz * 5 * (Px // 2) * math.log2(Px // 2)
    fft_y = 5 * Py * math.log2(Py)                               # flops of one complex column transform
    out = {"rows_fwd": {"bytes": state + (wl.N * 4 if ms0_per_cell else 0) + U, "flops": fl_rows},
           "rows_inv": {"bytes": U + state, "flops": fl_rows}}
    if lp:
        tensor = (4 + 6 * (wl.nz - 1)) * Cx * Py * 4
        out["columns"] = {"bytes": 2 * U + tensor, "flops": 3 * wl.nz * Cx * 2 * fft_y + Cx * Py * wl.nz * wl.nz * 36}
    else:
        T = 3 * Pz * Cx * wl.ny * 8
        tensor = (4 if wl.nz == 1 else 6) * (Pz // 2 + 1) * Cx * Py * 4
        out["columns"] = {"bytes": (U + T if wl.nz > 1 else 2 * T) + tensor,
                          "flops": 3 * Pz * Cx * 2 * fft_y + Pz * Cx * Py * (20 if wl.nz == 1 else 36)}
        if wl.nz > 1:
            out["z_inverse"] = {"bytes": T + U, "flops": 3 * Cx * wl.ny * 8 * wl.nz * (Pz - 1)}
    return out


def source_hash():
    """Identity of the kernels a measurement belongs to: sha256 over the library's sources and the build script."""
    import hashlib
    h = hashlib.sha256()
    base = os.path.join(ROOT, "paper_2106_05593_b200")
    files = sorted(os.path.join(base, "csrc", f) for f in os.listdir(os.path.join(base, "csrc")))
    for f in files + [os.path.join(base, "build.py"), os.path.join(ROOT, "include", "mmc.h")]:
        with open(f, "rb") as fh:
            h.update(os.path.basename(f).encode() + b"\0" + fh.read())
    return h.hexdigest()[:16]


_KERNEL_OF = (("colour_pass", "colour_pass_kernel"), ("rows_fwd", "demag_rows_fwd_kernel"), ("rows_inv", "demag_rows_inv_kernel"),
              ("columns", "demag_columns_kernel"), ("z_inverse", "demag_z_inverse_kernel"))


def ncu_traffic(cfg):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch (mean over the captured launches) of every kernel of the
    step, from the committed ncu capture profiles/traffic_cfg<N>.csv -- but only if profiles/traffic_cfg<N>.md says that the
    capture was taken from exactly these sources (source_hash); otherwise there is no measurement and the field is null."""
    import csv
    md = os.path.join(ROOT, "profiles", f"traffic_cfg{cfg}.md"); cs = os.path.join(ROOT, "profiles", f"traffic_cfg{cfg}.csv")
    if not (os.path.exists(md) and os.path.exists(cs)):
        return {}
    with open(md) as f:
        if f"source_hash: {source_hash()}" not in f.read():
            return {}
    per = {}
    with open(cs) as f:
        rows = [ln for ln in f if ln.startswith('"')]
    rd = csv.DictReader(rows)
    for r in rd:
        kind = {"dram__bytes_read.sum": "dram_bytes", "dram__bytes_write.sum": "dram_bytes",
                "sm__inst_executed.sum": "warp_instructions"}.get(r["Metric Name"])
        if kind is None:
            continue
        v = float(r["Metric Value"].replace(",", "")) * {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(r["Metric Unit"], 1.0)
        name = next((k for pat, k in _KERNEL_OF if pat in r["Kernel Name"]), None)
        if name:
            d = per.setdefault(name, {}).setdefault(kind, {}); d[r["ID"]] = d.get(r["ID"], 0.0) + v
    return {k: {kind: sum(d.values()) / len(d) for kind, d in kinds.items()} for k, kinds in per.items()}


def replica_seed(base_seed: int, rank: int) -> int:
    """Independent replica per rank: distinct Philox key, same workload."""
    return (int(base_seed) + 0x9E3779B97F4A7C15 * int(rank)) & 0xFFFFFFFFFFFFFFFF


def aggregate_over_ranks(units: float, seconds: float, backend_device: str = "cuda") -> float:
    """value = units of all ranks / max-over-ranks time (the contract's whole-job aggregate)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return units / seconds
    t = torch.tensor([units], dtype=torch.float64, device=backend_device)
    s = torch.tensor([seconds], dtype=torch.float64, device=backend_device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    dist.all_reduce(s, op=dist.ReduceOp.MAX)
    return float(t.item() / s.item())


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index=0):
        self.rows = []; self.proc = None; self.gpu = gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.gpu)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True); self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.rows.append(ln.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            p = [x.strip() for x in r.split(",")]
            if len(p) < 9:
                continue
            try:
                sm.append(float(p[1])); mx.append(float(p[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), p[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def _workload(cfg: int, small: bool, shape=None):
    import workloads as W
    if shape:                                     # same recipe on another mesh (the L2-exceeding stand-in); not a bench line
        dims = [int(x) for x in shape.split(",")]
        kw = dict(nx=dims[0], ny=dims[1])
        if len(dims) > 2 and cfg in (4, 6):
            kw["nz"] = dims[2]
        return W.make(cfg, **kw)
    if small:
        kw = {1: {}, 2: dict(nx=64, ny=64), 3: dict(nx=64, ny=64), 4: dict(nx=64, ny=64, nz=4), 5: dict(nx=140, ny=140),
              6: dict(nx=64, ny=64, nz=4)}[cfg]
        return W.make(cfg, **kw)
    return W.make(cfg)


# ------------------------------------------------------------------------------------------------ oracle arm
def oracle_sample(cfg: int):
    """Bounded sample of config `cfg` for the CPU legs: same recipe, reduced mesh."""
    import workloads as W
    kw = {1: {}, 2: {}, 3: dict(nx=256, ny=256), 4: dict(nx=256, ny=256, nz=4), 5: dict(nx=560, ny=560),
          6: dict(nx=128, ny=128, nz=10)}[cfg]
    return W.make(cfg, **kw), kw


def _omp_threads(n=None):
    """Thread count of the OpenMP runtime the oracle's C file was built against (libgomp): set it (n) or read it back.
    The oracle itself is not touched: this is the runtime's own switch, like the OMP_NUM_THREADS environment variable."""
    import ctypes
    try:
        omp = ctypes.CDLL("libgomp.so.1")
        if n is not None:
            omp.omp_set_num_threads(int(n))
        return int(omp.omp_get_max_threads())
    except OSError:
        return int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))


def time_oracle(cfg: int, steps, warmup: int, threads=None, budget_s=10.0):
    """The fp64 oracle as it stands on a bounded sample of config `cfg`: whole iterations (updates/s) and, separately, its
    demag convolution (numpy.fft on the padded grid, not a tuned FFT).  threads=None: all host cores."""
    import oracle as O
    import workloads as W
    wl, kw = oracle_sample(cfg)
    wl.adaptive_cone = False
    o = O.OracleMMC(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, wl.pbc_mask, store_fp32=True)
    W.configure(o, wl, O.Material)
    all_cores = os.cpu_count() or 1
    cores = _omp_threads(threads if threads else all_cores)
    conv = None
    if wl.demag:
        o.demag_field()                       # tensor set-up outside the timed region (as on the GPU side)
        t0 = time.perf_counter(); n = 0
        while n < 3 or (time.perf_counter() - t0 < 1.0 and n < 50):
            o.demag_field(); n += 1
        conv = n / (time.perf_counter() - t0)
    t0 = time.perf_counter()
    o.run(max(1, warmup))
    per = (time.perf_counter() - t0) / max(1, warmup)
    if steps is None:                         # cpu_baseline leg: about budget_s of CPU work
        steps = int(min(400, max(2, round(budget_s / max(per, 1e-3)))))
    t0 = time.perf_counter()
    o.run(steps)
    dt = time.perf_counter() - t0
    _omp_threads(all_cores)
    sample = f"{wl.name} recipe on a {wl.nx}x{wl.ny}x{wl.nz} mesh ({wl.n_active} non-empty cells), {steps} iterations incl. numpy.fft demag"
    return {"value": wl.n_active * steps / dt, "seconds": dt, "steps": steps, "cores": cores, "sample": sample,
            "demag_convolutions_per_sec": conv}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    steps = max(1, args.steps); warm = max(1, args.warmup)
    r = time_oracle(args.config, steps, warm)
    v, dt, cores, sample = r["value"], r["seconds"], r["cores"], r["sample"]
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": steps, "warmup": warm,
            "ms_per_step": 1e3 * dt / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": f"cfg{args.config} (oracle sample: {sample})"},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "demag_convolutions_per_sec": r["demag_convolutions_per_sec"]},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1")); rank = int(os.environ.get("RANK", "0")); local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    import paper_2106_05593_b200 as P
    import workloads as W
    cfg = args.config
    wl = _workload(cfg, args.small, args.shape)
    wl.adaptive_cone = False                      # fixed cone/sigma for throughput runs (SURVEY 8(d) timing protocol)
    wl.seed = replica_seed(wl.seed, rank)
    g = P.MMC(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, wl.pbc_mask, device=local)
    W.configure(g, wl, P.Material)
    K, Wm = max(1, args.steps), max(3, args.warmup)
    dev = torch.device("cuda", local)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    g.sweep(Wm)                                   # warm-up (also builds the demag plan and tensor spectrum)
    barrier()
    sampler = ClockSampler(local); sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()                                   # the ctx runs on torch's current stream, where these events are recorded
    g.sweep(K)                                    # EXACTLY K iterations, enqueued back to back: the timed region of `value`
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    # per-kernel device times: a second pass with CUDA events around every launch (the events add a little idle time
    # between kernels, which is why the headline above is timed without them)
    Kp = min(K, 50)
    phases = g.sweep_timed(Kp)
    phases = {k: v * (K / Kp) for k, v in phases.items()}      # scaled to K so that the per-step divisions below hold
    clocks = sampler.stop()
    units = float(wl.n_active) * K
    value = aggregate_over_ranks(units, ms * 1e-3)
    ob = g.observables()

    # e2e through the C ABI with HOST buffers (mmc_set_m_host / mmc_get_m_host do the copies on the ctx stream): pinned
    # H2D of the step's m, one iteration, D2H of m and of the read-out struct
    nE = max(3, min(K, 20))
    host_in = [torch.from_numpy(np.ascontiguousarray(wl.m0[a])).pin_memory() for a in range(3)]
    host_out = [torch.empty(wl.N, dtype=torch.float32).pin_memory() for _ in range(3)]
    L = P.lib()
    obs = P.Obs()

    def e2e_step():
        g._ck(L.mmc_set_m_host(g._h, host_in[0].data_ptr(), host_in[1].data_ptr(), host_in[2].data_ptr()))
        g._ck(L.mmc_sweep(g._h, 1))
        g._ck(L.mmc_get_m_host(g._h, host_out[0].data_ptr(), host_out[1].data_ptr(), host_out[2].data_ptr()))
        g._ck(L.mmc_get_observables(g._h, P.C.byref(obs)))      # synchronises; D2H of the read-out struct

    e2e_step(); barrier()
    t0 = time.perf_counter()
    for _ in range(nE):
        e2e_step()
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_val = aggregate_over_ranks(float(wl.n_active) * nE, e2e_s)
    h2d = 3 * wl.N * 4; d2h = 3 * wl.N * 4 + P.C.sizeof(P.Obs)
    # how much of an e2e step is the two copies (same calls, no iteration and no read-out in between)
    barrier()
    t0 = time.perf_counter()
    for _ in range(nE):
        g._ck(L.mmc_set_m_host(g._h, host_in[0].data_ptr(), host_in[1].data_ptr(), host_in[2].data_ptr()))
        g._ck(L.mmc_get_m_host(g._h, host_out[0].data_ptr(), host_out[1].data_ptr(), host_out[2].data_ptr()))
        torch.cuda.synchronize(dev)
    copies_s = (time.perf_counter() - t0) / nE

    if rank == 0:
        peak, peak_src = _peaks()
        step_ms = sum(phases.values()) / K
        percell, mask, ms0_pc = layout_flags(wl)
        # per-launch time, algorithmic bytes and flops of every kernel of the step (CUDA events on the ctx stream)
        kern = {}
        pass_ms = (phases["red"] + phases["black"]) / (2 * K)
        bpu = pass_bytes_per_update(wl)
        kern["colour_pass_kernel"] = {"launch_ms": pass_ms, "launches_per_step": 2, "bytes": bpu * wl.n_active / 2.0,
                                      "units_per_launch": wl.n_active / 2.0, "bytes_per_unit": bpu}
        if wl.demag:
            db = demag_kernel_bytes(wl, ms0_pc)
            for name, ph in (("rows_fwd", "rows_fwd"), ("columns", "columns"), ("z_inverse", "z_inverse"), ("rows_inv", "rows_inv")):
                if name not in db:
                    continue
                kern["demag_" + name + "_kernel"] = {"launch_ms": phases[ph] / K, "launches_per_step": 1, "bytes": db[name]["bytes"],
                                                    "flops": db[name]["flops"], "units_per_launch": wl.N,
                                                    "bytes_per_unit": db[name]["bytes"] / wl.N}
        full = not args.small and not args.shape
        traffic = ncu_traffic(cfg) if full else {}          # measured by ncu from exactly these sources, or nothing
        ISSUE_PEAK = 148 * 4 * 1.965e9                      # warp instructions / s (B200_PROFILING.md: 148 SMs, 1965 MHz; 4 schedulers per SM)
        FMA_PEAK = 74.4                                     # TFLOP/s: 148 SM x 128 FP32 lanes x 2 flop x 1.965 GHz (no tensor cores: no contraction here)
        for k, d in kern.items():
            t = d["launch_ms"] * 1e-3
            d["achieved_GBs"] = d["bytes"] / t / 1e9 if t > 0 else 0.0
            d["frac_of_hbm_peak"] = d["achieved_GBs"] / peak
            d["share_of_step"] = d["launch_ms"] * d["launches_per_step"] / step_ms if step_ms > 0 else None
            tr = traffic.get(k, {})
            d["ncu_traffic_bytes"] = tr.get("dram_bytes")
            d["ncu_warp_instructions"] = tr.get("warp_instructions")
            if "flops" in d:
                d["achieved_TFLOPs"] = d["flops"] / t / 1e12 if t > 0 else 0.0
                d["frac_of_fma_peak"] = d["achieved_TFLOPs"] / FMA_PEAK
            if tr.get("warp_instructions") and t > 0:
                d["issue_slot_frac"] = tr["warp_instructions"] / t / ISSUE_PEAK
            # which roofline is the tighter one for this kernel: the larger of the HBM fraction (algorithmic bytes) and the
            # plain-ALU fraction (algorithmic flops for the transforms; issue slots, from the ncu instruction count, for the pass)
            alu = max([x for x in (d.get("frac_of_fma_peak"), d.get("issue_slot_frac")) if x is not None], default=None)
            d["bound"] = "alu" if (alu is not None and alu > d["frac_of_hbm_peak"]) else "hbm"
        dom = max(kern, key=lambda k: kern[k]["launch_ms"])          # the dominant kernel = longest single launch
        dk = kern[dom]
        demag_ms = sum(phases[k] for k in ("pack", "rows_fwd", "columns", "rows_inv", "z_inverse")) / K
        # launches inside the timed region (graph nodes are kernel launches too); small meshes without demag: ONE launch runs all K iterations
        single_launch = (not wl.demag) and wl.N <= 8192 and not percell
        per_iter = (len([k for k in kern if k.startswith("demag_")]) * wl.demag_updates if wl.demag else 0) + 3
        roof_hbm = {"kernel": dom, "bound": "hbm", "achieved": dk["achieved_GBs"], "peak": peak, "unit": "GB/s",
                    "frac": dk["frac_of_hbm_peak"], "traffic": dk["ncu_traffic_bytes"], "peak_source": peak_src,
                    "algorithmic_bytes_per_unit": dk["bytes_per_unit"], "units_per_launch": dk["units_per_launch"],
                    "launch_ms": dk["launch_ms"], "share_of_step": dk["share_of_step"],
                    "traffic_source": (f"profiles/traffic_cfg{cfg}.csv (ncu, source_hash {source_hash()})" if dk["ncu_traffic_bytes"] is not None
                                       else "no ncu capture of these sources: null")}
        roof_alu = None
        if "achieved_TFLOPs" in dk:
            roof_alu = {"kernel": dom, "bound": "alu", "achieved": dk["achieved_TFLOPs"], "peak": FMA_PEAK, "unit": "TFLOP/s",
                        "frac": dk["frac_of_fma_peak"], "issue_slot_frac": dk.get("issue_slot_frac"), "traffic": dk["ncu_traffic_bytes"],
                        "peak_source": "derived: 148 SM x 128 lanes x 2 flop x 1.965 GHz (B200_PROFILING.md unit counts and clocks); "
                                       "algorithmic flops = 5 n log2 n per complex transform + the tensor products",
                        "launch_ms": dk["launch_ms"], "share_of_step": dk["share_of_step"]}
        elif "issue_slot_frac" in dk:
            roof_alu = {"kernel": dom, "bound": "alu", "achieved": dk["ncu_warp_instructions"] / (dk["launch_ms"] * 1e-3) / 1e12,
                        "peak": ISSUE_PEAK / 1e12, "unit": "T warp-instr/s", "frac": dk["issue_slot_frac"], "traffic": dk["ncu_traffic_bytes"],
                        "peak_source": "derived: 148 SM x 4 schedulers x 1.965 GHz; instructions from the ncu capture",
                        "launch_ms": dk["launch_ms"], "share_of_step": dk["share_of_step"]}
        primary, other = (roof_alu, roof_hbm) if (dk["bound"] == "alu" and roof_alu) else (roof_hbm, roof_alu)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm, "ms_per_step": ms / K,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{wl.name} {wl.nx}x{wl.ny}x{wl.nz} ({wl.n_active} non-empty cells)", "cfg": cfg,
                       "step": "1 MMC iteration = demag FFT convolution (rows, columns + tensor multiply, inverse rows) + red + "
                               "black colour pass + bookkeeping",
                       "l2": "inputs larger than L2: state + B_d + class words + FFT work array + tensor spectrum = "
                             f"{(kern.get('demag_columns_kernel', {'bytes': 0})['bytes'] + 7 * 4 * wl.N) / 1e6:.0f} MB streamed per step "
                             "(L2 = 126 MB)" if wl.N >= 2 ** 22 else
                             "working set fits L2 (small config, a parity case rather than a bench line)",
                       "parallelism": "replicas" if world > 1 else "single GPU", "cone_deg": wl.cone_deg,
                       "acceptance": ob["accepted"] / max(1, ob["trials"]),
                       "launch_path": ("one launch of the single-CTA kernel for all K iterations" if single_launch else
                                       "first iteration as plain launches, the rest replayed from CUDA graphs of 16 and 1 iterations")},
            "clocks": clocks,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": nE,
                    "ms_per_step": 1e3 * e2e_s / nE, "copies_ms_per_step": 1e3 * copies_s,
                    "copies_share_of_step": copies_s / (e2e_s / nE) if e2e_s > 0 else None},
            "gpu_launches": 1 if single_launch else per_iter * K,
            "phases_ms_per_step": {k: v / K for k, v in phases.items()},
            "phases_path": ("mmc_sweep_timed: launch-per-kernel with CUDA events around every launch" +
                            ("; NOT the path of `value`, which runs the single-launch small-mesh kernel" if single_launch else
                             "; same kernels as `value`, which replays them from CUDA graphs without the events")),
            "sweep_only_updates_per_sec": wl.n_active / (2 * pass_ms * 1e-3) if pass_ms > 0 else None,
            "demag_convolutions_per_sec": (1e3 / demag_ms) if (wl.demag and demag_ms > 0) else None,
            "roofline": primary,
            "roofline_other": other,
            "kernels": kern,
        }
        if not args.no_cpu_baseline and world == 1:
            # the oracle beside it: all host cores (~10 s) and one core (~6 s), plus its convolutions/s
            r = time_oracle(cfg, None, 1, None, 10.0)
            r1 = time_oracle(cfg, None, 1, 1, 6.0)
            line["cpu_baseline"] = {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"],
                                    "demag_convolutions_per_sec": r["demag_convolutions_per_sec"],
                                    "one_core": {"value": r1["value"], "cores": r1["cores"], "sample": r1["sample"],
                                                 "demag_convolutions_per_sec": r1["demag_convolutions_per_sec"]}}
        print(json.dumps(line))
    g.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=400)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5, 6],
                    help="BASELINE.json config (default 4: the largest fully magnetic mesh, 1024x1024x4)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--small", action="store_true", help="reduced mesh (debugging only; not a bench number)")
    ap.add_argument("--shape", default=None, help="nx,ny[,nz]: the config's recipe on another mesh (exploration; not a bench number)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
