#!/usr/bin/env python
"""bench.py -- cell-updates/s of the full DNSLABIB Navier-Stokes step (fp64) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4] [--piter P]

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


def oracle_rate(case_small, steps, warmup=0):
    """cell-updates/s of the CPU oracle as it stands, on a bounded sample."""
    import numpy as np
    from oracle import dnsref
    o = dnsref.Oracle(case_small["shape"], case_small["d"], case_small["nu"], case_small["alpha_c"], case_small["dt"],
                      mask=case_small["mask"], sources=case_small["sources"], body=case_small["body"],
                      n_piter=case_small["n_piter"])
    o.set_fields(case_small["u"], case_small["v"], case_small["w"], case_small["c"])
    if warmup:
        o.step(warmup)
    t = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t
    n = int(np.prod(case_small["shape"]))
    return n * steps / dt, dt / steps, dnsref.num_threads()


def run_reference(args):
    """--impl reference: the oracle (this tier's reference arm) timed on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_2204_02107_b200 import cases
    small = cases.config(args.config, shrink=2 if args.config >= 3 else 1)
    if args.piter:
        small["n_piter"] = args.piter
    steps = max(1, min(args.steps, 3))
    warm = 1 if args.warmup > 0 else 0
    rate, sec, cores = oracle_rate(small, steps, warm)
    sample = f"{small['name']} (config {args.config} generator at half resolution), P={small['n_piter']}, " \
             f"{steps} timed steps after {warm} warm-up, OpenMP over outer loops"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warm, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config {args.config}: {small['name']} room grid, P={small['n_piter']} (bounded sample "
                               f"of the 512x256x128 workload; CPU oracle, not a GPU run)"},
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
    breakdown = {k: {"ms_per_step": v[0] / K, "launches_per_step": v[1] / K,
                     "GBps_canonical": cb[k] * N / (v[0] / v[1] * 1e-3) / 1e9,
                     "GBps_moved": mv[k] * N / (v[0] / v[1] * 1e-3) / 1e9} for k, v in prof.items()}
    traffic = None
    tfile = os.path.join(ROOT, "profiles", "traffic.csv")   # class,case,dram bytes per launch (ncu --set full)
    if os.path.exists(tfile):
        for line in open(tfile):
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 3 and f[0] == dom and f[1] == case["name"]:
                traffic = float(f[2])
    step_bytes = (canonical_bytes_per_cell(P, masked) + (cb["filter"] if args.flags & 1 else 0.0)) * N
    step_gbs = step_bytes / (ms_max / K * 1e-3) / 1e9

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
            "config": {"workload": f"config {args.config}: {case['name']} ({N} cells), n_piter={P}, "
                                   f"{'masked room with inlet source' if masked else 'periodic box'}",
                       "grid": list(case["shape"][::-1]), "n_piter": P, "flags": args.flags,
                       "l2": "working set 19 fields x %.0f MB >> 126 MB L2, no flush needed" % (8 * N / 1e6),
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "gpu_launches": launches,
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 5 * 8 * N, "d2h_bytes_per_step": 5 * 8 * N,
                    "steps": Ke, "note": "dnslab_set_fields(host) + dnslab_step(1) + dnslab_get_fields(host) per step, "
                                         "pinned buffers"},
            "roofline": {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                         "bytes_per_cell_per_launch": cb[dom], "share_of_step": d_ms / tot_ms,
                         "moved_bytes_per_cell_per_launch": mv[dom], "achieved_moved": achieved_moved,
                         "frac_moved": achieved_moved / peak, "near_solid_fraction": fb,
                         "timing": "CUDA events around every launch (dnslab_profile), separate pass of K steps",
                         "note": "achieved/frac count SURVEY.md 8(d)'s canonical bytes (the fixed denominator; 65 RK field passes "
                                 "per step); this implementation moves fewer (48), so frac can exceed 1 -- achieved_moved/"
                                 "frac_moved count the bytes it really moves, and traffic is ncu's DRAM bytes per launch"},
            "step_roofline": {"canonical_bytes_per_cell": canonical_bytes_per_cell(P, masked), "achieved": step_gbs,
                              "peak": peak, "unit": "GB/s", "frac": step_gbs / peak},
            "kernels": breakdown,
        }
    s.close()
    del s
    torch.cuda.empty_cache()

    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            from paper_2204_02107_b200 import cases
            small = cases.config(args.config, shrink=2 if args.config >= 3 else 1)
            small["n_piter"] = P
            rate, sec, cores = oracle_rate(small, 3)
            out["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                                   "sample": f"{small['name']} (config {args.config} generator at half resolution), "
                                             f"P={P}, 3 steps, {sec:.2f} s/step"}
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config number (1-5)")
    ap.add_argument("--piter", type=int, default=0, help="override n_piter (0 = the config's own)")
    ap.add_argument("--flags", type=int, default=0, help="dnslab_params_t.flags (1: eq. 6 filter, 2: per-stage projection, "
                                                         "8: two-stage RK kernel); the headline line uses 0")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs only)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
