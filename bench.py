#!/usr/bin/env python
"""bench.py — throughput of the cooling step (BASELINE.json metric: Gcell-updates/s and achieved
HBM GB/s on one B200).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c5|c5u|c2|c3|c4-<n>|s512]
                    [--variant auto|global|smem|tex_point|tex_hwfilter|analytic] [--impl ours|reference]

A "step" is one cool_apply over the whole batch (every row of SURVEY.md §8(a): load, coordinates,
table retrieval, process combination, Coulomb exchange, limiter, sub-steps, store, luminosity).
Default workload c5 = BASELINE.json configs[4]: 512^3 cells fp32, three 48^4 process tables,
Coulomb coefficient table 48^2, 4 sub-steps, luminosity diagnostic, on the MAD-like field of
configs[2] resampled to 512^3 (north_star: "measured on synthetic MAD-like cell fields").
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2505_08855_b200 import synth  # noqa: E402  (numpy only)

METRIC = "Gcell-updates/s of the cooling step"
UNIT = "Gcell-updates/s"
SPEC_HBM_GBS = 8000.0                     # BASELINE.json: "vs 8 TB/s"
FALLBACK_HBM_GBS = 6650.0                 # B200_PROFILING.md fallback
# issue-slot ceiling of the SMs (the bound that actually limits the sub-stepped 4-D step): 148 SMs x 4 schedulers x
# 1 warp instruction per clock at clocks.max.sm 1965 MHz (B200_PROFILING.md unit counts) = 1163 G warp-instructions/s
ISSUE_PEAK_GWINST = 148 * 4 * 1.965
# dram__bytes and smsp__inst_executed per launch of the dominant kernel are read from profiles/r02_ncu_per_launch.csv
# (ncu_value below), the summary of the ncu captures kept under profiles/


# ------------------------------------------------------------------------------------------------
# workloads
# ------------------------------------------------------------------------------------------------
def workload_spec(name: str):
    """-> dict(label, table n, nc, nsub, dt, field recipe, diag, vol)."""
    if name == "c5":
        return dict(label="configs[4]: 512^3 fp32 MAD-like field, 3x48^4 tables + 48^2 Coulomb, nsub=4, luminosity",
                    n=[48, 48, 48, 48], nc=[48, 48], nsub=4, dt=1e-3, field=("mad", 512, 512, 512), diag=True, vol=True)
    if name == "c5u":
        return dict(label="configs[4] with log-uniform (worst-locality) cells: 512^3 fp32, 3x48^4 tables, nsub=4, luminosity",
                    n=[48, 48, 48, 48], nc=[48, 48], nsub=4, dt=1e-3, field=("logu", 512 ** 3, 5, 0.0), diag=True, vol=False)
    if name == "c2":
        return dict(label="configs[1]: 256^3 fp32 log-uniform with 1% outliers, table 128^3, single update",
                    n=[128, 128, 128], nc=[64, 64], nsub=1, dt=1e-3, field=("logu", 256 ** 3, 2, 0.01), diag=False, vol=False)
    if name == "c3":
        return dict(label="configs[2]: MAD-like 288x192x144 fp32, table 128^3, floor on, single update",
                    n=[128, 128, 128], nc=[64, 64], nsub=1, dt=1e-3, field=("mad", 288, 192, 144), diag=True, vol=True, floor=0.1)
    if name.startswith("c4-"):
        m = int(name[3:])
        return dict(label=f"configs[3]: 2^26 fp32 log-uniform cells, table {m}^3, single update",
                    n=[m, m, m], nc=[64, 64], nsub=1, dt=1e-3, field=("logu", 1 << 26, 4, 0.0), diag=False, vol=False)
    if name == "s512":
        return dict(label="512^3 fp32 MAD-like field, single update, table 128^3 + 64^2 Coulomb (3-D step of configs[2] at 512^3)",
                    n=[128, 128, 128], nc=[64, 64], nsub=1, dt=1e-3, field=("mad", 512, 512, 512), diag=False, vol=False)
    if name == "s512d":
        return dict(label="s512 with the luminosity diagnostic and volume weights", n=[128, 128, 128], nc=[64, 64], nsub=1, dt=1e-3,
                    field=("mad", 512, 512, 512), diag=True, vol=True)
    if name == "s512f":
        return dict(label="s512 with luminosity, volume weights and the temperature floor (the 3-D step of configs[2] at 512^3)",
                    n=[128, 128, 128], nc=[64, 64], nsub=1, dt=1e-3, field=("mad", 512, 512, 512), diag=True, vol=True, floor=0.1)
    raise SystemExit(f"unknown workload {name}")


def make_fields(spec, rank=0):
    f = spec["field"]
    if f[0] == "mad":
        return synth.mad_like_cells(f[1], f[2], f[3], dtype=np.float32, config=3 + 16 * rank)
    return synth.log_uniform_cells(f[1], dtype=np.float32, config=f[2] + 16 * rank, outlier_frac=f[3])


def table_ranges(n):
    rng = {0: synth.LOG_RHO, 1: synth.LOG_THETA, 2: synth.LOG_BSQ, 3: synth.LOG_THETA}
    nd = len(n)
    return list(range(nd)), [rng[a][0] for a in range(nd)], [rng[a][1] for a in range(nd)]


def bytes_per_cell(spec):
    return 24 + (4 if spec.get("vol") else 0) + (4 if spec.get("floor") else 0)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (measured copy bandwidth)"
    return FALLBACK_HBM_GBS, "fallback 6.65 TB/s of B200_PROFILING.md (MEASURED_PEAKS.json absent)"


# ------------------------------------------------------------------------------------------------
# oracle legs (cpu_baseline and --impl reference): the only places bench.py touches oracle/
# ------------------------------------------------------------------------------------------------
def oracle_leg(spec, desc, data, coul, fields, sample_cells, steps=1, scheme="explicit", nthreads=0):
    import oracle as O
    O.build()
    nd = desc.ndim
    otab = O.Table([desc.axis[k] for k in range(nd)], [desc.n[k] for k in range(nd)], [desc.lo[k] for k in range(nd)],
                   [desc.hi[k] for k in range(nd)], data, coul=coul, clo=[desc.clo[0], desc.clo[1]], chi=[desc.chi[0], desc.chi[1]])
    u = desc.units
    un = O.Units(u.rho_scale_cgs, u.mbh_msun, u.gamma_e, u.gamma_i, u.ln_lambda, u.ion_theta_mass_ratio, u.hth_cm, u.r_ref_rg, u.spin)
    cores = nthreads or O.max_threads()
    ncell = fields["rho"].size
    m = min(sample_cells, ncell)
    lo = (ncell - m) // 2                     # contiguous sample from the middle of the field
    sl = slice(lo, lo + m)
    times = []
    for _ in range(steps):
        t0 = time.perf_counter()
        step = O.step_implicit if scheme == "implicit" else O.step
        step(otab, un, fields["rho"][sl], fields["bsq"][sl], fields["theta_e"][sl], fields["theta_i"][sl], spec["dt"],
             nsub=spec["nsub"], h_floor=spec.get("floor", 0.0), r=fields["r"][sl] if spec.get("floor") else None,
             vol=fields["vol"][sl] if spec.get("vol") else None, nthreads=cores)
        times.append(time.perf_counter() - t0)
    return m, cores, times


# ------------------------------------------------------------------------------------------------
class ClocksMonitor:
    """SM clock and clock-event reasons sampled DURING the timed region (B200_PROFILING.md, clocks line).  The timed region
    of the default run is ~80 ms, shorter than nvidia-smi's start-up, so the samples come from NVML (the library nvidia-smi
    reads) on a thread of this process, every 2 ms; `nvidia-smi -lms` is the fallback when NVML cannot be loaded."""
    REASONS = (("hw_slowdown", 0x8), ("hw_thermal_slowdown", 0x40), ("sw_thermal_slowdown", 0x20), ("sw_power_cap", 0x4))

    def __init__(self, uuid):
        self.rows, self.max_mhz, self.source = [], None, None
        self._stop, self._thread, self._proc, self._path = threading.Event(), None, None, None
        try:
            import pynvml
            pynvml.nvmlInit()
            uuid = str(uuid)
            uuid = uuid if uuid.startswith("GPU-") else "GPU-" + uuid
            try:
                self._h = pynvml.nvmlDeviceGetHandleByUUID(uuid)
            except Exception:
                self._h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode())
            self._nv = pynvml
            self._reasons = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or pynvml.nvmlDeviceGetCurrentClocksThrottleReasons
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
            self._sample()                       # fails here, not on the thread, if the queries are not supported
            self.rows.clear()
            self.source = "nvml"
        except Exception:
            self._nv = None

    def _sample(self):
        nv = self._nv
        self.rows.append((float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)), int(self._reasons(self._h))))

    def _run(self):
        while not self._stop.is_set():
            try:
                self._sample()
            except Exception:
                break
            self._stop.wait(0.002)

    def start(self, gpu_index):
        if self._nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
            return
        f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self._path = f.name
        q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
            "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
        try:
            self._proc = subprocess.Popen(["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "20"],
                                          stdout=f, stderr=subprocess.DEVNULL)
            self.source = "nvidia-smi"
            t0 = time.time()                     # wait for its first row so that the timed region is covered
            while time.time() - t0 < 5.0 and os.path.getsize(self._path) == 0:
                time.sleep(0.01)
        except OSError:
            self._proc = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=self.max_mhz, reasons=[], samples=0, source=self.source)
        if self._thread is not None:
            self._stop.set()
            self._thread.join(timeout=2)
            if self.rows:
                out["sm_mhz"] = float(np.median([r[0] for r in self.rows])); out["samples"] = len(self.rows)
                out["sm_min_mhz"] = float(min(r[0] for r in self.rows))
                bits = 0
                for r in self.rows:
                    bits |= r[1]
                out["reasons"] = [nm for nm, b in self.REASONS if bits & b]
            return out
        if self._proc is not None:
            self._proc.terminate()
            try:
                self._proc.wait(timeout=5)
            except Exception:
                self._proc.kill()
        try:
            rows = [r.strip().split(",") for r in open(self._path) if r.strip()]
            rows = [r for r in rows if len(r) >= 7]
            if rows:
                sm = [float(r[0]) for r in rows]
                out["sm_mhz"] = float(np.median(sm)); out["sm_min_mhz"] = float(min(sm)); out["sm_max_mhz"] = float(rows[0][1]); out["samples"] = len(sm)
                for k, (nm, _) in enumerate(self.REASONS):
                    if any(r[3 + k].strip().lower().startswith("active") for r in rows):
                        out["reasons"].append(nm)
        except Exception:
            pass
        finally:
            try:
                if self._path:
                    os.unlink(self._path)
            except OSError:
                pass
        return out


def run_radpress(args, rank, local_rank, world):
    """--workload rp512: the radiation-pressure temperature correction (eq 29) on a 512^3 fp32 thick-disc
    field: one streaming kernel per step, 16 B/cell (rho, Theta_e, H read; Theta_e written).  Not the default line."""
    metric, unit = "Gcell/s of the radiation-pressure temperature correction (eq 29)", "Gcell/s"
    label = "512^3 fp32 thick-disc field (synth.thick_disc_cells), tau_crit = 1 (Fig. 9(b))"
    tau_crit = 1.0
    if args.impl == "reference":
        if rank != 0:
            return 0
        import oracle as O
        O.build()
        f = synth.thick_disc_cells(512, 512, 16)
        un = O.Units()
        times = []
        for k in range(min(args.warmup, 1) + args.steps):
            t0 = time.perf_counter()
            O.radpress(un, f["rho"], f["theta_e"], f["hscale"], tau_crit)
            if k >= min(args.warmup, 1):
                times.append(time.perf_counter() - t0)
        m, tot = f["rho"].size, float(np.sum(times))
        val = m * args.steps / tot / 1e9
        print(json.dumps(dict(metric=metric, value=val, unit=unit, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                              ms_per_step=1e3 * tot / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                              data="synthetic", impl="reference", config=dict(workload="rp512", description=label, cells_per_step=m,
                                                                              note="oracle Part C (bisection, one host thread) on a phi-slab of the workload"),
                              cpu_baseline=dict(value=val, unit=unit, cores=1, kind="oracle", sample=f"{m} cells (a 512x512x16 phi-slab) per step"),
                              e2e=dict(value=val, unit=unit, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)))
        return 0
    import torch
    from paper_2505_08855_b200 import api
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    f = synth.thick_disc_cells(512, 512, 512, config=6 + 16 * rank)
    ncell = f["rho"].size
    keys = ("rho", "theta_e", "hscale")
    host = {k: torch.from_numpy(f[k]).pin_memory() for k in keys}
    d = {k: host[k].to(dev) for k in keys}
    out = torch.empty_like(d["theta_e"])
    d_cnt = torch.zeros(1, dtype=torch.int64, device=dev)
    units = api.default_units()
    stream = torch.cuda.current_stream().cuda_stream

    def step():
        api.cool_radpress_correct(units, ncell, api.COOL_F32, d["rho"], d["theta_e"], d["hscale"], tau_crit, out, d_cnt, stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    mon = ClocksMonitor(torch.cuda.get_device_properties(dev).uuid) if rank == 0 else None
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    if mon is not None:
        mon.start(local_rank)
    ev[0].record()
    for k in range(args.steps):
        step()
        ev[k + 1].record()
    barrier()
    clocks = mon.stop() if rank == 0 else None
    per_step_ms = np.array([ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)])
    total_ms = float(ev[0].elapsed_time(ev[-1]))
    # end to end: pinned host arrays in, corrected Theta_e and the counter out, every step
    h_out = torch.empty(ncell, dtype=torch.float32).pin_memory()
    e2e_steps = max(1, min(args.steps, 3))

    def hstep():
        for k in keys:
            d[k].copy_(host[k], non_blocking=True)
        step()
        h_out.copy_(out, non_blocking=True)
        return int(d_cnt.item())
    hstep()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        ncorr = hstep()
    barrier()
    dt_e2e = time.perf_counter() - t0
    if world > 1:
        t = torch.tensor([total_ms, dt_e2e], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms, dt_e2e = float(t[0].item()), float(t[1].item())
        dist.destroy_process_group()
    if rank != 0:
        return 0
    peak, peak_src = peaks()
    kern_ms = float(np.mean(per_step_ms))
    achieved = 16 * ncell / (kern_ms * 1e-3) / 1e9
    value = ncell * world * args.steps / (total_ms * 1e-3) / 1e9
    line = dict(metric=metric, value=value, unit=unit, n_gpus=world, steps=args.steps, warmup=args.warmup, ms_per_step=total_ms / args.steps,
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32", data="synthetic",
                config=dict(workload="rp512", description=label, cells_per_gpu=ncell, tau_crit=tau_crit, corrected_cells=ncorr,
                            l2="inputs (%.2f GB per step) larger than L2" % (12 * ncell / 1e9)),
                clocks=clocks, gpu_launches=args.steps,
                e2e=dict(value=ncell * world * e2e_steps / dt_e2e / 1e9, unit=unit, h2d_bytes_per_step=12 * ncell, d2h_bytes_per_step=4 * ncell + 8,
                         steps=e2e_steps, api="cool_radpress_correct after 3 pinned host->device copies, device->host copy of the result"),
                roofline=dict(bound="hbm", achieved=achieved, peak=peak, unit="GB/s", frac=achieved / peak,
                              traffic=ncu_value("rp512", "radpress", "dram_bytes"),
                              kernel="cool_radpress_kernel<float, VEC=1, COUNT=1>", bytes_per_cell=16, algorithmic_bytes_per_launch=16 * ncell,
                              peak_source=peak_src, ms_per_launch_median=float(np.median(per_step_ms)), ms_per_launch_best=float(per_step_ms.min())))
    if not args.no_cpu_baseline:
        import oracle as O
        O.build()
        sl = slice(ncell // 2, ncell // 2 + (1 << 23))
        t0 = time.perf_counter()
        O.radpress(O.Units(), f["rho"][sl], f["theta_e"][sl], f["hscale"][sl], tau_crit)
        t1 = time.perf_counter() - t0
        line["cpu_baseline"] = dict(value=(1 << 23) / t1 / 1e9, unit=unit, cores=1, kind="oracle",
                                    sample=f"{1 << 23} contiguous cells from the middle of the workload, one pass, {t1:.1f} s")
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------
# the paper's own table: --workload p100 and the App. A replay --workload appA-<N>
# ------------------------------------------------------------------------------------------------
CGS_AX = [4, 5, 6, 7]                                  # log H_th[cm], log B[G], log n_e[cm^-3], log T_e[K]
CGS_LO, CGS_HI = [3.0, 0.0, 2.0, 2.0], [12.0, 10.0, 25.0, 15.0]
CGS_C3LO, CGS_C3HI = [2.0, 2.0, 2.0], [25.0, 15.0, 15.0]


def run_cgs(args, rank, local_rank, world):
    """p100: one cooling step of 2^26 log-uniform cells (random radii) on the paper's 100^4 table (400 MB: beyond L2) and its
    100^3 Coulomb table.  appA-<N>: the paper's stand-alone test: N^4 lookups on a regular grid of
    (H_th, B, n_e, T_e), hardware-filtered texture (the paper's scheme) | point texture | global memory | analytic, as one
    cooling step per query cell (Coulomb off, dt -> 0: the lookup is all that differs between the variants)."""
    import torch
    from paper_2505_08855_b200 import api
    if args.impl == "reference":
        if rank == 0:
            print(json.dumps(dict(impl="reference", unavailable="the oracle leg for the paper's 100^4 table lives in tests/test_cgs_gpu.py (sampled cells); no timed CPU arm for this workload")))
        return 0
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    ntab = args.table_n
    desc = api.make_desc(CGS_AX, [ntab] * 4, CGS_LO, CGS_HI, 1, nc3=[ntab] * 3, c3lo=CGS_C3LO, c3hi=CGS_C3HI)
    t0 = time.perf_counter()
    data = api.cool_table_build_device(desc, device=local_rank)
    t_build = time.perf_counter() - t0
    _, coul3 = api.cool_table_build_host(api.make_desc(CGS_AX, [2] * 4, CGS_LO, CGS_HI, 0, nc3=[ntab] * 3, c3lo=CGS_C3LO, c3hi=CGS_C3HI), want_coulomb=True)
    table = api.cool_table_create(desc, data, coul3, device=local_rank)
    app = args.workload.startswith("appA-")
    g = torch.Generator(device=dev); g.manual_seed(20250508 + rank)
    MP, C, KB, ME = 1.67262192369e-24, 2.99792458e10, 1.380649e-16, 9.1093837015e-28
    rg, rs = 1.32712440018e26 * 10.0 / C ** 2, 3e-7
    if app:
        N = int(args.workload[5:])
        ncell = N ** 4
        idx = torch.arange(ncell, device=dev, dtype=torch.int64)
        frac = lambda k: ((idx // (N ** k)) % N).to(torch.float64) / (N - 1)            # k = 0: T_e fastest (the paper's flattening)
        Te = 10.0 ** (7.0 + 4.0 * frac(0)); ne = 10.0 ** (8.0 + 12.0 * frac(1)); B = 10.0 ** (1.0 + 7.0 * frac(2)); H = 10.0 ** (7.0 + 4.0 * frac(3))
        the = Te * KB / (ME * C * C); thi = the
        p = (the + thi) * (ME / MP)
        cs = torch.sqrt((5.0 / 3.0) * p / (1.0 + 2.5 * p))
        r = torch.clamp(H / (rg * cs) - 0.9375, min=1.0) ** (2.0 / 3.0)
        d = dict(rho=(ne * MP / rs), bsq=(B * B / (4.0 * np.pi * rs * C * C)), theta_e=the, theta_i=thi, r=r)
        d = {k: v.to(torch.float32) for k, v in d.items()}
        del idx, Te, ne, B, H, the, thi, p, cs, r
        label = f"App. A replay: {N}^4 = {ncell} lookups on a regular (H_th, B, n_e, T_e) grid, table {ntab}^4, one cooling step per query (Coulomb off)"
        dt, coul = 1e-6, api.COOL_COULOMB_OFF
    elif args.workload == "p100w":
        # queries spread over the WHOLE table (log-uniform in B, n_e, T_e over the paper's ranges, radii over four decades so
        # that H_th = c_s/Omega_K spreads too): unphysical as a simulation state, but the one workload whose table reads
        # do not stay inside an L2-resident corner of the 400 MB table
        ncell = 1 << 26
        u64 = lambda lo, hi: 10.0 ** (lo + (hi - lo) * torch.rand(ncell, device=dev, generator=g, dtype=torch.float64))
        ne, B, Te = u64(CGS_LO[2], CGS_HI[2]), u64(CGS_LO[1], CGS_HI[1]), u64(CGS_LO[3], CGS_HI[3])
        the = Te * KB / (ME * C * C)
        d = dict(rho=ne * MP / rs, bsq=B * B / (4.0 * np.pi * rs * C * C), theta_e=the, theta_i=the, r=u64(0.0, 4.0))
        d = {k: v.to(torch.float32) for k, v in d.items()}
        del ne, B, Te, the
        label = f"2^26 fp32 cells log-uniform over the WHOLE (B, n_e, T_e) range of the paper's {ntab}^4 table ({4 * ntab ** 4 / 1e6:.0f} MB), radii 1-10^4 r_g, single update"
        dt, coul = 1e-3, api.COOL_COULOMB_TABLE
    else:
        ncell = 1 << 26
        u = lambda lo, hi: 10.0 ** (lo + (hi - lo) * torch.rand(ncell, device=dev, generator=g, dtype=torch.float32))
        d = dict(rho=u(-6.0, 0.0), bsq=u(-8.0, 0.0), theta_e=u(-3.0, 1.5), theta_i=u(-3.0, 1.5), r=u(0.2, 2.8))
        label = f"2^26 fp32 log-uniform cells with log-uniform radii, the paper's {ntab}^4 table ({4 * ntab ** 4 / 1e6:.0f} MB) + {ntab}^3 Coulomb table, single update"
        dt, coul = 1e-3, api.COOL_COULOMB_TABLE
    the_o = torch.empty(ncell, dtype=torch.float32, device=dev); thi_o = torch.empty_like(the_o)
    stream = torch.cuda.current_stream().cuda_stream
    names = ["tex_hwfilter", "tex_point", "global"] + (["analytic"] if app and args.with_analytic else []) if (app or args.variant == "auto") else [args.variant]
    res = {}
    mon = ClocksMonitor(torch.cuda.get_device_properties(dev).uuid)
    mon.start(local_rank)
    for nm in names:
        params = api.make_params(dt, 1, 0.3, 0.0, api.VARIANTS[nm], coul)
        step = lambda: api.cool_apply(table, ncell, api.COOL_F32, d["rho"], d["bsq"], d["theta_e"], d["theta_i"], the_o, thi_o, params, r=d["r"], stream=stream)
        steps = args.steps if nm != "analytic" else max(1, min(args.steps, 2))
        for _ in range(args.warmup if nm != "analytic" else 1):
            step()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            step()
        e1.record(); torch.cuda.synchronize()
        res[nm] = dict(ms_per_step=float(e0.elapsed_time(e1)) / steps, kernel=api.cool_last_kernel_name())
    clocks = mon.stop()
    peak, peak_src = peaks()
    best = "global" if "global" in res else names[0]
    ms = res[best]["ms_per_step"]
    bpc = 28                                                     # rho, bsq, Theta_e, Theta_i, r read; Theta_e', Theta_i' written
    ach = bpc * ncell / (ms * 1e-3) / 1e9
    line = dict(metric=METRIC, value=ncell / (ms * 1e-3) / 1e9, unit=UNIT, n_gpus=1, steps=args.steps, warmup=args.warmup, ms_per_step=ms,
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=args.workload, description=label, cells_per_gpu=ncell, variant=best, table_build_s_on_device=t_build,
                            l2="inputs (%.2f GB per step) and the table larger than L2" % (bpc * ncell / 1e9)),
                variants=res, clocks=clocks, gpu_launches=args.steps,
                roofline=dict(bound="hbm", achieved=ach, peak=peak, unit="GB/s", frac=ach / peak, traffic=ncu_value(args.workload, best, "dram_bytes"),
                              kernel=res[best]["kernel"], bytes_per_cell=bpc, algorithmic_bytes_per_launch=bpc * ncell, peak_source=peak_src,
                              note="algorithmic bytes are the cell stream; the 16 table corners of a cell are 16 scattered 32-byte sectors when the "
                                   "table does not fit L2 (see traffic)"))
    if "tex_hwfilter" in res and "global" in res:
        line["texture_over_global_time"] = res["tex_hwfilter"]["ms_per_step"] / res["global"]["ms_per_step"]
    if "analytic" in res:
        line["analytic_over_texture_time"] = res["analytic"]["ms_per_step"] / res["tex_hwfilter"]["ms_per_step"]
    print(json.dumps(line))
    table.destroy()
    return 0


def ncu_value(workload, variant, column):
    """Per-launch counters of the dominant kernel from the ncu captures summarised in profiles/r02_ncu_per_launch.csv
    (workload,variant,kernel,dram_bytes,warp_inst,source); None when that (workload, variant) was not captured."""
    path = os.path.join(ROOT, "profiles", "r02_ncu_per_launch.csv")
    if not os.path.exists(path):
        return None
    import csv
    with open(path) as fh:
        for row in csv.DictReader(fh):
            if row["workload"] == workload and row["variant"] == variant and row.get(column):
                return float(row[column])
    return None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c5")
    ap.add_argument("--variant", default="auto")
    ap.add_argument("--scheme", default="explicit", choices=["explicit", "implicit"], help="PAPER.md L185: (i) limiter or (ii) implicit solver")
    ap.add_argument("--shells", action="store_true", help="also compute the radial luminosity profile (eq 25) in the same launch (MAD-like workloads with diagnostics)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="skip the companion s512 measurement of the default workload")
    ap.add_argument("--cpu-sample", type=int, default=1 << 27)
    ap.add_argument("--table-n", type=int, default=100, help="points per axis of the paper's table (p100, appA-<N>); the paper uses 100")
    ap.add_argument("--with-analytic", action="store_true", help="appA-<N>: also time the analytic variant (slow)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                                       # timing rule: W >= 3

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.workload == "rp512":
        return run_radpress(args, rank, local_rank, world)
    if args.workload in ("p100", "p100w") or args.workload.startswith("appA-"):
        return run_cgs(args, rank, local_rank, world)
    spec = workload_spec(args.workload)
    axis, lo, hi = table_ranges(spec["n"])

    # ---------------- reference arm: the oracle on host cores, rank 0 only ----------------------
    if args.impl == "reference":
        if rank != 0:
            return 0
        # tables from the oracle's own fillers: this arm loads nothing of the product
        import oracle as O
        O.build()
        un0 = O.Units()
        if len(spec["n"]) == 3:
            data = [O.fill_total3(un0, spec["n"], lo, hi)]
        else:
            data = O.fill_proc4(un0, spec["n"], lo, hi)
        coul = O.fill_coulomb2(un0, spec["nc"], [synth.LOG_THETA[0]] * 2, [synth.LOG_THETA[1]] * 2)

        class _Desc:                                   # what oracle_leg reads of a table descriptor
            pass
        desc = _Desc()
        desc.ndim = len(spec["n"]); desc.axis = axis; desc.n = spec["n"]; desc.lo = lo; desc.hi = hi
        desc.clo = [synth.LOG_THETA[0]] * 2; desc.chi = [synth.LOG_THETA[1]] * 2; desc.units = un0
        small = dict(spec); f = spec["field"]
        if f[0] == "mad":
            small["field"] = ("mad", f[1], f[2], max(1, (1 << 22) // (f[1] * f[2])))   # a phi-slab of the same field
        else:
            small["field"] = ("logu", min(f[1], 1 << 22), f[2], f[3])
        fields = make_fields(small)
        sample = min(fields["rho"].size, 1 << 22)
        for _ in range(min(args.warmup, 1)):
            oracle_leg(spec, desc, data, coul, fields, sample, 1, args.scheme)
        m, cores, times = oracle_leg(spec, desc, data, coul, fields, sample, args.steps, args.scheme)
        tot = float(np.sum(times))
        val = m * args.steps / tot / 1e9
        line = dict(metric=METRIC, value=val, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                    ms_per_step=1e3 * tot / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None,
                    dtype="f64", data="synthetic", impl="reference",
                    config=dict(workload=args.workload, description=spec["label"], cells_per_step=m,
                                note="oracle (oracle/cool_oracle.c, gcc -O2, OpenMP) on a bounded contiguous sample of the workload"),
                    cpu_baseline=dict(value=val, unit=UNIT, cores=cores, kind="oracle", sample=f"{m} contiguous cells of the workload per step"),
                    e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
        print(json.dumps(line))
        return 0

    # ---------------- our arm ---------------------------------------------------------------------
    import torch
    from paper_2505_08855_b200 import api
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    desc = api.make_desc(axis, spec["n"], lo, hi, 1 if len(spec["n"]) == 3 else 3, nc=spec["nc"],
                         clo=[synth.LOG_THETA[0]] * 2, chi=[synth.LOG_THETA[1]] * 2)
    data, coul = api.cool_table_build_host(desc, want_coulomb=True)
    table = api.cool_table_create(desc, data, coul, device=local_rank)
    variant = api.VARIANTS[args.variant]
    resolved = table.auto_variant() if variant == api.COOL_V_AUTO else variant

    fields = make_fields(spec, rank)          # weak scaling: every rank owns a full batch (cells are independent)
    ncell = fields["rho"].size
    keys = ["rho", "bsq", "theta_e", "theta_i"] + (["vol"] if spec.get("vol") else []) + (["r"] if spec.get("floor") else [])
    host = {k: torch.from_numpy(fields[k]).pin_memory() for k in keys}
    d = {k: host[k].to(dev, non_blocking=True) for k in keys}
    the_o = torch.empty(ncell, dtype=torch.float32, device=dev)
    thi_o = torch.empty(ncell, dtype=torch.float32, device=dev)
    d_diag = torch.zeros(api.DIAG_BYTES, dtype=torch.uint8, device=dev) if spec["diag"] else None
    scheme = api.COOL_SCHEME_IMPLICIT if args.scheme == "implicit" else api.COOL_SCHEME_EXPLICIT
    params = api.make_params(spec["dt"], spec["nsub"], 0.3, spec.get("floor", 0.0), variant, api.COOL_COULOMB_TABLE, scheme)
    stream = torch.cuda.current_stream().cuda_stream
    shell_cells, lum_shell = 0, None
    if args.shells:
        if spec["field"][0] != "mad" or not spec["diag"]:
            raise SystemExit("--shells needs a MAD-like workload with diagnostics (c5, c3, s512d, s512f)")
        shell_cells = spec["field"][2] * spec["field"][3]                      # all (theta, phi) cells of one radial index
        lum_shell = torch.zeros(4 * spec["field"][1], dtype=torch.float64, device=dev)

    def step():
        api.cool_apply(table, ncell, api.COOL_F32, d["rho"], d["bsq"], d["theta_e"], d["theta_i"], the_o, thi_o, params,
                       r=d.get("r"), vol=d.get("vol"), d_diag=d_diag, stream=stream, shell_cells=shell_cells, lum_shell=lum_shell)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    launches_per_step = api.cool_last_launch_count()
    kernel_name = api.cool_last_kernel_name()         # the dispatcher's own choice, reported by the library
    barrier()
    mon = ClocksMonitor(torch.cuda.get_device_properties(dev).uuid) if rank == 0 else None
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    if mon is not None:
        mon.start(local_rank)
    ev[0].record()
    for k in range(args.steps):
        step()
        ev[k + 1].record()
    barrier()
    clocks = mon.stop() if rank == 0 else None
    per_step_ms = np.array([ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)])
    total_ms = float(ev[0].elapsed_time(ev[-1]))
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    value = ncell * world * args.steps / (total_ms * 1e-3) / 1e9
    diag_out = None
    if d_diag is not None:
        dd = api.cool_diag.from_buffer_copy(d_diag.cpu().numpy().tobytes()).as_dict()
        if world > 1:                           # the only cross-rank datum: 4 luminosity sums
            t = torch.tensor([dd["lum_total"], dd["lum_brems"], dd["lum_synch"], dd["lum_compton"]], dtype=torch.float64, device=dev)
            dist.all_reduce(t)
            dd["lum_total"], dd["lum_brems"], dd["lum_synch"], dd["lum_compton"] = [float(x) for x in t.tolist()]
        diag_out = dd

    # ---- executed sub-steps (outside the timed region).  A cell stops sub-stepping as soon as a sub-step changes no bit of its
    # state (exact: every later sub-step would be the same identity).  Measured through the public call: chain nsub single
    # sub-step updates with h = dt/nsub and count, stage by stage, the cells every earlier stage has changed. ----
    substeps_executed = None
    if spec["nsub"] > 1 and args.scheme == "explicit" and not args.shells:
        p1 = api.make_params(spec["dt"] / spec["nsub"], 1, 0.3, spec.get("floor", 0.0), variant, api.COOL_COULOMB_TABLE, scheme)
        cur_e, cur_i = d["theta_e"].clone(), d["theta_i"].clone()
        nxt_e, nxt_i = torch.empty_like(cur_e), torch.empty_like(cur_i)
        active = torch.ones(ncell, dtype=torch.bool, device=dev)
        executed = 0
        for _ in range(spec["nsub"]):
            executed += int(active.sum().item())
            api.cool_apply(table, ncell, api.COOL_F32, d["rho"], d["bsq"], cur_e, cur_i, nxt_e, nxt_i, p1, r=d.get("r"), vol=d.get("vol"), stream=stream)
            torch.cuda.synchronize()
            active &= (nxt_e.view(torch.int32) != cur_e.view(torch.int32)) | (nxt_i.view(torch.int32) != cur_i.view(torch.int32))
            cur_e, nxt_e = nxt_e, cur_e
            cur_i, nxt_i = nxt_i, cur_i
        substeps_executed = executed / ncell
        del cur_e, cur_i, nxt_e, nxt_i, active
        step()
        torch.cuda.synchronize()

    # ---- companion lines of the default workload, same timing protocol: (1) the single-update 3-D step (table 128^3) on the
    # same 512^3 field, which is what north_star's 70 % bar is about; (2) configs[4] on log-uniform cells (worst locality),
    # "run both" ----
    also = None
    if args.workload == "c5" and args.variant == "auto" and not args.no_also and args.scheme == "explicit":
        also = []
        peak2, _ = peaks()

        def timed(fn):
            for _ in range(args.warmup):
                fn()
            barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(args.steps):
                fn()
            e1.record()
            barrier()
            ms = float(e0.elapsed_time(e1)) / args.steps
            if world > 1:
                t = torch.tensor([ms], dtype=torch.float64, device=dev)
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
                ms = float(t.item())
            return ms
        spec2 = workload_spec("s512")
        axis2, lo2, hi2 = table_ranges(spec2["n"])
        desc2 = api.make_desc(axis2, spec2["n"], lo2, hi2, 1, nc=spec2["nc"], clo=[synth.LOG_THETA[0]] * 2, chi=[synth.LOG_THETA[1]] * 2)
        data2, coul2 = api.cool_table_build_host(desc2, want_coulomb=True)
        table2 = api.cool_table_create(desc2, data2, coul2, device=local_rank)
        params2 = api.make_params(spec2["dt"], 1, 0.3, 0.0, api.COOL_V_AUTO, api.COOL_COULOMB_TABLE)
        ms2 = timed(lambda: api.cool_apply(table2, ncell, api.COOL_F32, d["rho"], d["bsq"], d["theta_e"], d["theta_i"], the_o, thi_o, params2, stream=stream))
        ach2 = 24 * ncell / (ms2 * 1e-3) / 1e9
        also.append(dict(workload="s512", description=spec2["label"], ms_per_step=ms2, value=ncell * world / (ms2 * 1e-3) / 1e9, unit=UNIT,
                         gpu_launches_per_step=api.cool_last_launch_count(),
                         roofline=dict(bound="hbm", achieved=ach2, peak=peak2, unit="GB/s", frac=ach2 / peak2, traffic=ncu_value("s512", "global", "dram_bytes"),
                                       kernel=api.cool_last_kernel_name(), bytes_per_cell=24),
                         frac_of_8TBs=ach2 / SPEC_HBM_GBS))
        table2.destroy()
        spec3 = workload_spec("c5u")
        f3 = make_fields(spec3, rank)
        d3 = {k: torch.from_numpy(f3[k]).to(dev) for k in ("rho", "bsq", "theta_e", "theta_i")}
        del f3
        params3 = api.make_params(spec3["dt"], spec3["nsub"], 0.3, 0.0, api.COOL_V_AUTO, api.COOL_COULOMB_TABLE)
        ms3 = timed(lambda: api.cool_apply(table, ncell, api.COOL_F32, d3["rho"], d3["bsq"], d3["theta_e"], d3["theta_i"], the_o, thi_o, params3,
                                           d_diag=d_diag, stream=stream))
        ach3 = 24 * ncell / (ms3 * 1e-3) / 1e9
        also.append(dict(workload="c5u", description=spec3["label"], ms_per_step=ms3, value=ncell * world / (ms3 * 1e-3) / 1e9, unit=UNIT,
                         gpu_launches_per_step=api.cool_last_launch_count(),
                         roofline=dict(bound="hbm", achieved=ach3, peak=peak2, unit="GB/s", frac=ach3 / peak2, traffic=ncu_value("c5u", "global", "dram_bytes"),
                                       kernel=api.cool_last_kernel_name(), bytes_per_cell=24),
                         note="uncorrelated cells: bound by L2 -> L1 gather traffic and instruction issue, not by HBM"))
        del d3
        step()                                       # leave the_o / thi_o and d_diag holding the main workload's result for the e2e check below
        torch.cuda.synchronize()

    # ---- end to end: host buffers, copies inside the timed region (rank-local, max over ranks) ----
    e2e = None
    if not args.no_e2e:
        ho_e = torch.empty(ncell, dtype=torch.float32).pin_memory()
        ho_i = torch.empty(ncell, dtype=torch.float32).pin_memory()
        e2e_steps = max(1, min(args.steps, 3))

        def hstep():
            return api.cool_apply_host(table, ncell, api.COOL_F32, host["rho"], host["bsq"], host["theta_e"], host["theta_i"],
                                       ho_e, ho_i, params, r=host.get("r"), vol=host.get("vol"), want_diag=spec["diag"])
        hstep()
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            hstep()
        barrier()
        dt_e2e = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt_e2e], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt_e2e = float(t.item())
        e2e = dict(value=ncell * world * e2e_steps / dt_e2e / 1e9, unit=UNIT,
                   h2d_bytes_per_step=int(sum(host[k].numel() * 4 for k in keys)),
                   d2h_bytes_per_step=int(2 * ncell * 4 + (api.DIAG_BYTES if spec["diag"] else 0)),
                   steps=e2e_steps, api="cool_apply_host (C ABI, pinned host buffers, chunked copy/compute overlap)")
        same = bool(torch.equal(ho_e, the_o.cpu()) and torch.equal(ho_i, thi_o.cpu()))
        e2e["matches_device_path"] = same

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    peak, peak_src = peaks()
    bpc = bytes_per_cell(spec)
    kern_ms = float(np.mean(per_step_ms))                     # the step's kernels back to back (fp32 kernel + the precise pass where one runs)
    achieved = bpc * ncell / (kern_ms * 1e-3) / 1e9
    explicit = args.scheme == "explicit"
    vname = api.VARIANT_NAMES[resolved]
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
                ms_per_step=total_ms / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f32", data="synthetic",
                config=dict(workload=args.workload, description=spec["label"], cells_per_gpu=ncell, nsub=spec["nsub"],
                            variant=api.VARIANT_NAMES[resolved], scheme=args.scheme, radial_profile=bool(args.shells), l2="inputs (%.2f GB per step) larger than L2" % (bpc * ncell / 1e9),
                            cell_substeps_executed_per_update=substeps_executed,
                            substeps_note="nsub sub-steps per update are requested; a cell whose sub-step changes no bit stops early (exact); the executed count is measured by chaining single sub-step calls"),
                hbm_gbs=achieved * world, frac_of_8TBs=achieved / SPEC_HBM_GBS,
                clocks=clocks, e2e=e2e, gpu_launches=launches_per_step * args.steps,
                roofline=dict(bound="hbm", achieved=achieved, peak=peak, unit="GB/s", frac=achieved / peak,
                              traffic=(ncu_value(args.workload, vname, "dram_bytes") if explicit and not args.shells else None),
                              kernel=kernel_name, bytes_per_cell=bpc, algorithmic_bytes_per_launch=bpc * ncell, peak_source=peak_src,
                              ms_per_launch_median=float(np.median(per_step_ms)), ms_per_launch_best=float(per_step_ms.min())),
                diag=diag_out)
    winst = ncu_value(args.workload, vname, "warp_inst") if explicit and not args.shells else None
    if winst:
        gw = winst / (kern_ms * 1e-3) / 1e9
        line["issue_roofline"] = dict(bound="alu", achieved=gw, peak=ISSUE_PEAK_GWINST, unit="G warp-instructions/s", frac=gw / ISSUE_PEAK_GWINST,
                                      warp_inst_per_launch=winst,
                                      note="instruction-issue ceiling (148 SMs x 4 schedulers x 1965 MHz); instruction count of all kernels of a step from profiles/r02_ncu_per_launch.csv")
    if also is not None:
        line["also"] = also
    if not args.no_cpu_baseline:
        m, cores, times = oracle_leg(spec, desc, data, coul, fields, args.cpu_sample if explicit else min(args.cpu_sample, 1 << 23), 1, args.scheme)
        line["cpu_baseline"] = dict(value=m / times[0] / 1e9, unit=UNIT, cores=cores, kind="oracle",
                                    sample=f"{m} contiguous cells from the middle of the workload, one pass, {times[0]:.1f} s")
        m1, _, t1 = oracle_leg(spec, desc, data, coul, fields, min(args.cpu_sample, 1 << 22) if explicit else 1 << 19, 1, args.scheme, nthreads=1)
        line["cpu_baseline"]["single_thread"] = dict(value=m1 / t1[0] / 1e9, unit=UNIT, cores=1,
                                                     sample=f"{m1} contiguous cells from the middle of the workload, one pass, {t1[0]:.1f} s")
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
