#!/usr/bin/env python
"""bench.py -- cell-updates/s of the full DNSLABIB Navier-Stokes step (fp64) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4] [--piter P]
                  [--flags F] [--mode step|reductions|particles] [--traffic-csv profiles/<ncu raw export>.csv]

One "step" = one pass of the whole hot path (4 fused RHS+RK stages, divergence, P x FFT Poisson
iteration of eq. 9, projection) over the synthetic 512x256x128 room grid of BASELINE.json configs[3]
(the grid the target is quoted on).  N > 1 runs N independent replicas, one per GPU (DESIGN.md:
"replicas only" -- the path has no sharded form, so there is no collective), weak scaling.
Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "cell-updates/s per full NS step (fp64)"
UNIT = "cell-updates/s"


def canonical_bytes_per_cell(P, masked):
    """SURVEY.md 8(d) / DESIGN.md: B(P) = 8 (72 + 11 P) + (5 + P)/8; unmasked: no p^k read, no mask."""
    if masked:
        return 8.0 * (72 + 11 * P) + (5 + P) / 8.0
    return 8.0 * (72 + 10 * P)


# Bytes per cell per launch of each kernel class.
# "canonical": SURVEY.md 8(d)'s model (accumulate-form RK with Qc: 12+20+20+12 passes; div R3 W1; 5 FFT passes of
# R1 W1 per solve; dense p^k + mask read per eq. 9 iteration; projection R4 W3).
# "moved": what this implementation must move (Qc eliminated: 8+16+12+12 passes; eq. 9 only at the near-solid
# cells, a fraction fb of the grid: index 4 + saved d 8 + d 8 + p centre 8 + face 1 + ~1 neighbour 8 bytes).
def class_bytes_per_cell(masked, fb=0.0):
    m = 0.125 if masked else 0.0
    canonical = {
        "rk_stage": (96 + 160 + 160 + 96) / 4.0 + m,
        "div": 32.0,
        "fft_x": 16.0,
        "fft_y": 16.0,
        "fft_z_solve": 16.0,
        "fft_xy": 16.0,         # two-pass solve: x and the high digit of y (R1 W1 of the complex array, 8 B/cell each way)
        "fft_yz_solve": 16.0,   # two-pass solve: low digit of y, z, division, and back (R1 W1)
        "project": 56.0 + m,
        "eq9_sparse": 8.0 + m,
        "filter": 64.0 + m,
    }
    moved = dict(canonical)
    moved["rk_stage"] = (64 + 128 + 96 + 96) / 4.0 + (1.0 if masked else 0.0)   # stage 2 also writes S; stage 4 reads Q4, S
    moved["project"] = 56.0 + (1.0 if masked else 0.0)
    moved["eq9_sparse"] = 37.0 * fb
    moved["filter"] = 64.0 + (1.0 if masked else 0.0)
    return canonical, moved


def near_solid_fraction(mask):
    """Fraction of cells with at least one solid face neighbour (where eq. 9's bracket can be non-zero)."""
    import numpy as np
    if mask is None:
        return 0.0
    fluid = mask != 0
    allf = np.ones(mask.shape, dtype=bool)
    for ax in range(3):
        allf &= np.roll(fluid, 1, axis=ax) & np.roll(fluid, -1, axis=ax)
    return float(1.0 - allf.mean())


# kernel-class -> regular expression on ncu's demangled kernel name
CLASS_KERNELS = {
    "rk_stage": r"k_rk(_march)?<", "div": r"k_div", "fft_x": r"k_fft_x<", "fft_y": r"k_fft_col<", "fft_z_solve": r"k_fft_z_solve<",
    "fft_xy": r"k_fft_xy<", "fft_yz_solve": r"k_fft_yz_solve<",
    "project": r"k_project", "eq9_sparse": r"k_eq9", "filter": r"k_filter", "reduce": r"k_courant|k_box", "particles": r"k_particles",
}
_UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def ncu_traffic(path, cls, case):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum, mean over the captured launches) of the
    kernels of class `cls`, read from an `ncu --page raw --csv` export of a `--set full` capture of THIS workload
    (the .md beside the .csv names the command).  The export's grid sizes must be those of `case`, otherwise the
    capture belongs to another workload and the answer is None.  Returns (bytes or None, source note)."""
    import csv
    import re
    if not path:
        return None, "no ncu export given (--traffic-csv)"
    if not os.path.exists(path):
        return None, f"{os.path.relpath(path, ROOT)} not found"
    rows = list(csv.reader(open(path)))
    hdr, units, data = rows[0], rows[1], rows[2:]
    try:
        cn, cr, cw = hdr.index("Kernel Name"), hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
    except ValueError:
        return None, "export lacks dram__bytes_read.sum / dram__bytes_write.sum"
    pat = re.compile(CLASS_KERNELS.get(cls, cls))
    if units[cr] not in _UNIT or units[cw] not in _UNIT:
        return None, f"unknown unit {units[cr]!r} / {units[cw]!r} in {os.path.relpath(path, ROOT)}"
    vals = [float(r[cr]) * _UNIT[units[cr]] + float(r[cw]) * _UNIT[units[cw]] for r in data if pat.search(r[cn])]
    if not vals:
        return None, f"no {cls} kernel in {os.path.relpath(path, ROOT)}"
    # a capture of another grid is not this workload's traffic: the RK kernels' grids give the cell count away
    meta = os.path.splitext(path)[0] + ".md"
    if not os.path.exists(meta) or case["name"] not in open(meta).read():
        return None, f"{os.path.relpath(meta, ROOT)} does not name workload {case['name']}: the capture belongs to another workload"
    return sum(vals) / len(vals), f"{os.path.relpath(path, ROOT)}: mean of {len(vals)} launches"


def default_traffic_csv(args):
    """The committed `ncu --set full` export that belongs to this line's workload (profiles/<name>.md names the command
    and the workload); None if no capture of it is committed -- roofline.traffic is then null."""
    if args.mode == "reductions":
        name = "r03c_reductions_raw.csv" if args.config == 4 else None
    elif args.mode == "particles":
        name = "r03c_particles_raw.csv" if args.config == 4 else None
    else:
        name = {4: "r02e_ncu_full_raw.csv", 3: "r03c_c3_raw.csv", 5: "r03c_c5_raw.csv"}.get(args.config)
    return os.path.join(ROOT, "profiles", name) if name else None


def load_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled during the timed region."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def wait_ready(self, timeout=5.0):
        """Block until nvidia-smi has delivered its first row, so that a short timed region is still sampled."""
        t_end = time.time() + timeout
        while self.proc is not None and not self.rows and time.time() < t_end:
            time.sleep(0.02)

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        inside = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.2]
        rows = inside or [r for (_, r) in self.rows]
        sm, mx, reasons = [], [], set()
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        out = {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
               "reasons": sorted(reasons), "samples": len(sm), "samples_in_timed_region": len(inside)}
        if not inside:
            # nothing was sampled while the timed steps ran: what is reported is NOT the clock under load
            out["note"] = "no nvidia-smi sample fell inside the timed region; values are from outside it (use more --steps)"
        return out


def job_value(ms_local, n_cells, steps, world, device):
    """Whole-job cell-updates/s of `world` independent replicas: every rank advanced n_cells cells by
    `steps` steps; the job time is the MAX over ranks of the device-timed milliseconds (no data-path
    collective: DESIGN.md "replicas only").  Returns (value, ms_max)."""
    import torch
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_max = float(t.item())
    return world * n_cells * steps / (ms_max * 1e-3), ms_max


def make_case(cfg, piter):
    from paper_2204_02107_b200 import cases
    case = cases.config(cfg)
    if piter:
        case["n_piter"] = piter
    return case


def _omp_set_threads(n):
    """Thread count of the OpenMP runtime the oracle is linked against (the oracle's code is not touched)."""
    import ctypes
    from oracle import dnsref
    dnsref.lib()                                     # make sure libgomp is loaded
    ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))


def oracle_rate(case, steps, warmup=0, threads=None):
    """cell-updates/s of the CPU oracle as it stands, on `case`; threads=None: all host cores."""
    import numpy as np
    from oracle import dnsref
    all_cores = dnsref.num_threads()
    if threads:
        _omp_set_threads(threads)
    try:
        o = dnsref.Oracle(case["shape"], case["d"], case["nu"], case["alpha_c"], case["dt"], mask=case["mask"],
                          sources=case["sources"], body=case["body"], n_piter=case["n_piter"])
        o.set_fields(case["u"], case["v"], case["w"], case["c"])
        if warmup:
            o.step(warmup)
        t = time.perf_counter()
        o.step(steps)
        dt = time.perf_counter() - t
        used = dnsref.num_threads()
        o.close()
    finally:
        if threads:
            _omp_set_threads(all_cores)
    n = int(np.prod(case["shape"]))
    return n * steps / dt, dt / steps, used


def cpu_baseline(case, cfg):
    """The oracle beside the GPU number: on the bench workload itself, all host cores for 3 steps
    (1 step at config 5), and ONE thread for 1 step (config 5: the same generator at half resolution, said so)."""
    from paper_2204_02107_b200 import cases
    nall = 1 if cfg == 5 else 3
    rate, sec, cores = oracle_rate(case, nall)
    single_case, where = case, "the same workload"
    if cfg == 5:
        single_case, where = cases.config(5, shrink=2), "config 5's generator at half resolution (512x256x128)"
        single_case["n_piter"] = case["n_piter"]
    rate1, sec1, _ = oracle_rate(single_case, 1, threads=1)
    return {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{case['name']} itself, P={case['n_piter']}, {nall} steps on {cores} threads ({sec:.2f} s/step)",
            "single_thread": {"value": rate1, "unit": UNIT, "cores": 1,
                              "sample": f"{where}, 1 step on 1 thread ({sec1:.1f} s/step)"}}


def workload_name(config, case):
    """config.workload: the same string on the GPU arm and on the reference arm (the driver compares them)."""
    N = int(case["shape"][0]) * int(case["shape"][1]) * int(case["shape"][2])
    masked = case["mask"] is not None
    return (f"config {config}: {case['name']} ({N} cells), n_piter={case['n_piter']}, "
            f"{'masked room with inlet source' if masked else 'periodic box'}")


def run_reference(args):
    """--impl reference: the oracle (this tier's reference arm) timed on the host cores, on the bench workload
    itself (config 5: half resolution); every timed step is one oracle step; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_2204_02107_b200 import cases
    case = cases.config(args.config, shrink=2 if args.config == 5 else 1)
    if args.piter:
        case["n_piter"] = args.piter
    steps = max(1, min(args.steps, 5))
    warm = 1 if args.warmup > 0 else 0
    rate, sec, cores = oracle_rate(case, steps, warm)
    sample = f"{case['name']}" + (" (config 5's generator at half resolution)" if args.config == 5 else " itself") + \
             f", P={case['n_piter']}, {steps} timed steps after {warm} warm-up, {cores} threads (OpenMP over outer loops)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warm, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config, case), "grid": list(case["shape"][::-1]), "n_piter": case["n_piter"],
                   "arm": "CPU oracle on the host cores, not a GPU run; steps capped at 5"},
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2204_02107_b200 import binding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the DNSLAB path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    case = make_case(args.config, args.piter)
    N = int(np.prod(case["shape"]))
    P = case["n_piter"]
    masked = case["mask"] is not None
    s = binding.solver_for_case(case, device=f"cuda:{local}", flags=args.flags)
    K, W = args.steps, max(args.warmup, 3)

    # ---- device-resident timing: K steps, CUDA events on the solver's stream
    s.step(W)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.wait_ready()
    barrier()
    l0 = s.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    e0.record(s.stream)
    s.step(K)
    e1.record(s.stream)
    barrier()
    t1 = time.time()
    ms = e0.elapsed_time(e1)
    launches = s.launch_count() - l0
    clocks = sampler.stop(t0, t1) if sampler else None
    value, ms_max = job_value(ms, N, K, world, dev)

    # ---- per-kernel pass (same workload, K steps, events around every launch)
    s.profile(True)
    s.step(K)
    prof = s.profile_read()
    s.profile(False)
    fb = near_solid_fraction(case["mask"])
    cb, mv = class_bytes_per_cell(masked, fb)
    prof = {k: v for k, v in prof.items() if v[1] > 0}
    tot_ms = sum(v[0] for v in prof.values()) or 1.0
    dom = max(prof, key=lambda k: prof[k][0])
    d_ms, d_n = prof[dom]
    peak, peak_src = load_peak()
    achieved = cb[dom] * N / (d_ms / d_n * 1e-3) / 1e9
    achieved_moved = mv[dom] * N / (d_ms / d_n * 1e-3) / 1e9
    breakdown = {k: {"ms_per_step": v[0] / K, "launches_per_step": v[1] / K, "us_per_launch": v[0] / v[1] * 1e3,
                     "GBps_canonical": cb.get(k, 0.0) * N / (v[0] / v[1] * 1e-3) / 1e9,
                     "GBps_moved": mv.get(k, 0.0) * N / (v[0] / v[1] * 1e-3) / 1e9} for k, v in prof.items()}
    traffic, traffic_src = ncu_traffic(args.traffic_csv or default_traffic_csv(args), dom, case)
    step_bytes = (canonical_bytes_per_cell(P, masked) + (cb["filter"] if args.flags & 1 else 0.0)) * N
    step_gbs = step_bytes / (ms_max / K * 1e-3) / 1e9
    moved_step = sum(mv.get(k, 0.0) * v[1] / K for k, v in prof.items())   # bytes per cell per step actually required

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    Ke = max(1, min(K, args.e2e_steps))
    e2e_value = None
    if not args.no_e2e:
        host_in = {k: torch.from_numpy(case[k]).pin_memory() for k in "uvwc"}
        host_p = torch.zeros(case["shape"], dtype=torch.float64).pin_memory()
        host_out = {k: torch.empty(case["shape"], dtype=torch.float64).pin_memory() for k in "uvwcp"}
        for _ in range(2):
            s.set_fields(host_in["u"], host_in["v"], host_in["w"], host_in["c"], host_p)
            s.step(1)
            s.get_fields(**host_out)
        barrier()
        e0.record(s.stream)
        for _ in range(Ke):
            s.set_fields(host_in["u"], host_in["v"], host_in["w"], host_in["c"], host_p)
            s.step(1)
            s.get_fields(**host_out)
        e1.record(s.stream)
        barrier()
        e2e_value, _ = job_value(e0.elapsed_time(e1), N, Ke, world, dev)
        assert bool(torch.isfinite(host_out["u"]).all())

    out = None
    if rank == 0:
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config, case),
                       "grid": list(case["shape"][::-1]), "n_piter": P, "flags": args.flags,
                       "l2": "working set 19 fields x %.0f MB >> 126 MB L2, no flush needed" % (8 * N / 1e6),
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "gpu_launches": launches,
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 5 * 8 * N, "d2h_bytes_per_step": 5 * 8 * N,
                    "steps": Ke, "note": "dnslab_set_fields(host) + dnslab_step(1) + dnslab_get_fields(host) per step, "
                                         "pinned buffers"},
            "roofline": {"bound": "hbm", "kernel": dom, "achieved": achieved_moved, "peak": peak, "unit": "GB/s",
                         "frac": achieved_moved / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                         "bytes_per_cell_per_launch": mv[dom], "share_of_step": d_ms / tot_ms,
                         "canonical_bytes_per_cell_per_launch": cb[dom], "canonical_achieved": achieved,
                         "canonical_frac": achieved / peak, "near_solid_fraction": fb,
                         "timing": "CUDA events around every launch (dnslab_profile), separate pass of K steps",
                         "note": "achieved/frac count the algorithmic bytes of THIS kernel (DESIGN.md section 6: what it must "
                                 "move per cell and launch); canonical_* count SURVEY.md 8(d)'s model of the method (65 RK "
                                 "field passes per step where this implementation moves 48), kept for reference -- that "
                                 "figure can exceed 1; traffic is ncu's DRAM bytes per launch from the committed export"},
            "step_roofline": {"moved_bytes_per_cell": moved_step, "achieved": moved_step * N / (ms_max / K * 1e-3) / 1e9,
                              "frac": moved_step * N / (ms_max / K * 1e-3) / 1e9 / peak, "peak": peak, "unit": "GB/s",
                              "canonical_bytes_per_cell": canonical_bytes_per_cell(P, masked),
                              "canonical_achieved": step_gbs, "canonical_frac": step_gbs / peak,
                              "note": "whole step: bytes every kernel of the step must move (sum over the classes launched) "
                                      "over the step time; canonical_* = north_star's '% of the HBM roofline' on SURVEY.md "
                                      "8(d)'s byte model"},
            "kernels": breakdown,
        }
    s.close()
    del s
    torch.cuda.empty_cache()

    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            out["cpu_baseline"] = cpu_baseline(case, args.config)
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def run_extra(args):
    """--mode reductions | particles: bench lines for the NEXT-3 and NEXT-4 rows on the same workload.
    Not the headline: each line names its own metric.  Single GPU."""
    import numpy as np
    import torch
    from paper_2204_02107_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the DNSLAB path has no CPU fallback)")
    torch.cuda.set_device(0)
    case = make_case(args.config, args.piter)
    N = int(np.prod(case["shape"]))
    nz, ny, nx = case["shape"]
    masked = case["mask"] is not None
    peak, peak_src = load_peak()
    s = binding.solver_for_case(case, device="cuda:0")
    K, W = args.steps, max(args.warmup, 3)
    s.step(W)
    s.synchronize()
    sampler = ClockSampler(0)
    sampler.wait_ready()
    t0 = time.time()
    base = {"n_gpus": 1, "steps": K, "warmup": W, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic"}
    traffic, traffic_src = ncu_traffic(args.traffic_csv or default_traffic_csv(args),
                                       "k_courant" if args.mode == "reductions" else "particles", case)
    if args.mode == "reductions":
        # dnslab_courant: one streaming read of u, v, w (24 B/cell); dnslab_scalar_stats over the whole box: two
        # passes over c and the mask byte (2 x 9 B/cell).  Both calls synchronise; the device time is taken from the
        # library's per-class events (class "reduce").
        for _ in range(W):
            s.courant(); s.scalar_stats((0, 0, 0), (nx, ny, nz))
        l0 = s.launch_count()
        s.profile(True)
        for _ in range(K):
            s.courant()
        ms_co, n_co = s.profile_read()["reduce"]
        s.profile(True)
        for _ in range(K):
            s.scalar_stats((0, 0, 0), (nx, ny, nz))
        ms_st, n_st = s.profile_read()["reduce"]
        s.profile(False)
        launches = s.launch_count() - l0
        co_gbs = 24.0 * N / (ms_co / K * 1e-3) / 1e9
        st_gbs = (2 * 8.0 + (2.0 if masked else 0.0)) * N / (ms_st / K * 1e-3) / 1e9
        out = dict(base, metric="GB/s streamed by dnslab_courant (NEXT-3 reduction, 24 B/cell)", value=co_gbs, unit="GB/s",
                   ms_per_step=ms_co / K,
                   config={"workload": f"config {args.config}: {case['name']} ({N} cells); dnslab_courant and "
                                       f"dnslab_scalar_stats over the whole box, {K} calls each"},
                   gpu_launches=launches,
                   roofline={"bound": "hbm", "kernel": "reduce (k_courant)", "achieved": co_gbs, "peak": peak, "unit": "GB/s",
                             "frac": co_gbs / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src},
                   scalar_stats={"ms_per_call": ms_st / K, "GBps": st_gbs, "frac": st_gbs / peak,
                                 "bytes_per_cell": 2 * 8.0 + (2.0 if masked else 0.0), "launches_timed_per_call": n_st / K})
    else:
        # NEXT-4: n particles (default 10^6, 5-100 um droplets, uniformly seeded in the box) advanced after every step
        n = args.particles
        r = np.random.default_rng(77)
        L = np.array([nx * case["d"][0], ny * case["d"][1], nz * case["d"][2]])
        st = np.empty((8, n))
        st[0:3] = r.random((3, n)) * L[:, None]
        st[3:6] = 0.01 * r.standard_normal((3, n))
        st[6] = 5e-6 + 95e-6 * r.random(n)
        st[7] = 1000.0
        dev = torch.from_numpy(st).cuda()
        s.particles_attach(dev, 1.2, (0.0, 0.0, -9.81))
        s.step(W)
        l0 = s.launch_count()
        s.profile(True)
        s.step(K)
        prof = s.profile_read()
        s.profile(False)
        launches = s.launch_count() - l0
        ms_p, n_p = prof["particles"]
        tot = sum(v[0] for v in prof.values())
        rate = n * K / (ms_p * 1e-3)
        # per particle: 8 state doubles read, 6 written, 24 gathered field values (sector-granular in practice)
        gbs = (14 + 24) * 8.0 * n / (ms_p / K * 1e-3) / 1e9
        out = dict(base, metric="particle-updates/s (NEXT-4, eqs. 10-13, implicit Euler after every fluid step)", value=rate,
                   unit="particle-updates/s", ms_per_step=ms_p / K,
                   config={"workload": f"config {args.config}: {case['name']} ({N} cells) with {n} Lagrangian particles",
                           "particles": n},
                   gpu_launches=launches,
                   roofline={"bound": "hbm", "kernel": "particles (k_particles)", "achieved": gbs, "peak": peak, "unit": "GB/s",
                             "frac": gbs / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                             "note": "304 B per particle (8 state reads, 6 writes, 24 gathered velocities)"},
                   share_of_step=ms_p / tot, fluid_step_ms=(tot - ms_p) / K)
    s.synchronize()
    out["clocks"] = sampler.stop(t0, time.time())
    out["e2e"] = {"value": None, "unit": out["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                  "note": "not a headline line: the end-to-end figure is on the default --mode step line"}
    s.close()
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config number (1-5)")
    ap.add_argument("--piter", type=int, default=0, help="override n_piter (0 = the config's own)")
    ap.add_argument("--flags", type=int, default=0, help="dnslab_params_t.flags (1: eq. 6 filter, 2: per-stage projection); "
                                                         "the headline line uses 0")
    ap.add_argument("--mode", default="step", choices=["step", "reductions", "particles"],
                    help="step: the headline line; reductions / particles: the NEXT-3 / NEXT-4 lines")
    ap.add_argument("--particles", type=int, default=1000000, help="--mode particles: how many")
    ap.add_argument("--traffic-csv", default=None,
                    help="ncu --page raw --csv export of a --set full capture of this workload (roofline.traffic)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs only)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.mode != "step":
        run_extra(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
