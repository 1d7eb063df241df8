#!/usr/bin/env python
"""bench.py -- throughput of the B200-native MAC projection (one "step" = one whole projection:
face coefficients -> coarsening -> rhs -> V-cycles to 1e-10 -> velocity correction).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4N] [--n 512]
    python bench.py --impl reference ...      # the CPU oracle, as it stands, on the host cores

Prints ONE JSON line (rank 0).  `value` is level-0 cell-updates/s over the whole projection,
N^3 (nu_pre + nu_post) cycles / t(project), inputs resident in HBM;
`e2e` is the same metric through maestro_mac_project_host_seq() (K steps in one call, pinned HOST buffers, every step's
u, v, w copied host -> device and back inside the timed region, overlapped with the neighbouring steps' projections; the
unpipelined single call maestro_mac_project_host() is reported beside it).  `roofline` is the level-0 fused red-black smoother (k_rbgs_t2: the two sweeps of a smoothing step in
ONE pass over HBM): `achieved` = the bytes that pass must move (48 B per cell per launch: read phi, rhs, ax, ay, az, write phi;
DESIGN.md Sec. 6) over the mean device time of its launches, timed by CUDA event pairs inside the library on the call's stream
during the timed steps (desc.timing = 1); `per_sweep_*` restate it in SURVEY.md Sec. 8(d)'s per-sweep unit (48 B per cell per SWEEP).  Multi-GPU: replicas only:
every rank projects its own copy; value = all ranks' units / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "mac_projection_cell_updates_per_s"
UNIT = "cell-updates/s"
SMOOTHER_BYTES_PER_CELL = 48.0          # read phi, rhs, ax, ay, az; write phi (fp64)
FALLBACK_HBM_GBS = 6650.0               # /opt/skills/guides/B200_PROFILING.md fallback


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="4N", help="workload: 1, 2, 3N, 3D, 4N, 4D, 5 (BASELINE.json configs)")
    ap.add_argument("--n", type=int, default=512, help="cells per side")
    ap.add_argument("--smoother", type=int, default=0, help="0 two sweeps per HBM pass, TMA staging (default); 1 two-pass reference; 2 fused, cp.async staging; 3 fused, TMA 32x16 tile; 4 one sweep per pass, TMA staging")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the millisecond-scale configs 1, 2, 3N")
    ap.add_argument("--cpu-sample-n", type=int, default=0, help="cells per side of the oracle sample (0 = auto)")
    return ap.parse_args()


# ---- helpers ------------------------------------------------------------------------------------

def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(kernel: str, n: int):
    """dram bytes per launch of `kernel` at n^3 from the committed ncu summary, or None."""
    p = os.path.join(ROOT, "profiles", "roofline_traffic.csv")
    try:
        with open(p) as f:
            for line in f:
                parts = [x.strip() for x in line.split(",")]
                if len(parts) >= 3 and parts[0] == kernel and parts[1] == str(n):
                    return float(parts[2])
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (profiling recipe's clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.out = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=self.out, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        res = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return res
        try:
            self.proc.terminate()
            self.proc.wait(timeout=5)
        except Exception:
            try:
                self.proc.kill()
            except Exception:
                pass
        self.out.close()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            with open(self.path) as f:
                for line in f:
                    c = [x.strip() for x in line.split(",")]
                    if len(c) < 9:
                        continue
                    try:
                        sm.append(float(c[1])); mx.append(float(c[2])); pw.append(float(c[3]))
                    except ValueError:
                        continue
                    for nm, val in zip(names, c[5:9]):
                        if val.lower().startswith("active"):
                            reasons.add(nm)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            # "under load": samples whose power is within the upper half of the observed range
            lo, hi = min(pw), max(pw)
            load = [s for s, p in zip(sm, pw) if p >= lo + 0.5 * (hi - lo)] or sm
            res.update(sm_mhz=statistics.median(load), sm_max_mhz=max(mx), reasons=sorted(reasons),
                       samples=len(sm), power_w_max=hi)
        return res


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def host_mem_available_gb():
    try:
        with open("/proc/meminfo") as f:
            for line in f:
                if line.startswith("MemAvailable"):
                    return float(line.split()[1]) / 1e6
    except Exception:
        pass
    return 0.0


def cpu_oracle_run(config: str, n: int, threads: int = 0, wl=None):
    """One projection by the oracle on the host cores (threads = 0: all of them).  Returns (seconds, cycles, cells,
    threads used, sweeps per cycle)."""
    from oracle import mac_oracle as O
    from paper_1910_12979_b200 import workloads as W
    O.build()
    if threads > 0:
        O.set_num_threads(threads)
    else:
        O.set_num_threads(os.cpu_count() or 1)
    if wl is None:
        wl = W.by_name(config, n)
    g = O.make_grid(wl.n, wl.dx, wl.bc_lo, wl.bc_hi)
    b = O.make_base(wl.geometry, wl.nr, wl.dr, wl.center)
    mg = O.make_mg(nu_pre=wl.nu_pre, nu_post=wl.nu_post, max_cycles=wl.max_cycles, rel_tol=wl.rel_tol)
    u, v, w = wl.u.copy(), wl.v.copy(), wl.w.copy()
    t0 = time.perf_counter()
    status, _, stats = O.project(g, b, mg, wl.beta0, wl.rho0, wl.rho, u, v, w, wl.S, want_phi=False)
    dt = time.perf_counter() - t0
    assert status in (0, 1), status
    return dt, stats["cycles"], wl.ncells, O.num_threads(), (wl.nu_pre + wl.nu_post)


def workload_label(config: str, n: int) -> str:
    names = {"1": "config1 triply periodic", "2": "config2 planar atmosphere", "3N": "config3 star 1e4 (WALL)",
             "3D": "config3 star 1e4 (OUTFLOW)", "4N": "config4 star-in-a-box 1e6 (WALL x6, singular)",
             "4D": "config4 star-in-a-box 1e6 (OUTFLOW x6)", "5": "config5 convective shell"}
    return f"{names[config]} {n}^3 fp64, V(2,2) to 1e-10"


# ---- reference arm: the oracle, as it stands, on the host cores --------------------------------

def run_reference(a):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    ns = a.cpu_sample_n or 256                 # one projection at 256^3 is about 8 s on 16 cores
    ns = min(ns, a.n)
    for _ in range(a.warmup):
        cpu_oracle_run(a.config, ns)
    tot, units, cycles, threads = 0.0, 0.0, 0, 1
    for _ in range(a.steps):
        dt, cyc, cells, threads, nu = cpu_oracle_run(a.config, ns)
        tot += dt
        units += cells * nu * cyc
        cycles = cyc
    val = units / tot if tot > 0 else 0.0
    sample = f"{a.config} at {ns}^3 (same recipe as the {a.n}^3 workload), one full projection per step, {cycles} cycles"
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": a.gpus, "steps": a.steps,
        "warmup": a.warmup, "ms_per_step": 1e3 * tot / max(a.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_label(a.config, a.n) + f"; the reference arm times the oracle on the {ns}^3 instance of it",
                   "sample": sample, "same_config": ns == a.n},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                         "nproc": os.cpu_count(), "cpu_model": cpu_model()},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ---- our arm ------------------------------------------------------------------------------------

def aggregate_replicas(units_this_rank: float, t_dev_this_rank: float, world: int, device):
    """Replicas only: every rank projects its own copy.  Whole-job value = the units ALL ranks
    processed / the MAX over ranks of the device time.  Returns (value, t_max).  No data-path collective: one
    all_reduce(MAX) of the time and one all_reduce(SUM) of the unit count, after the timed region."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([t_dev_this_rank], dtype=torch.float64, device=device)
    n = torch.tensor([units_this_rank], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(n, op=dist.ReduceOp.SUM)
    t_max = float(t.item())
    return float(n.item()) / t_max, t_max


def run_ours(a):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1910_12979_b200 import build as B, mac, workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the MAC projection has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
    if rank == 0:
        B.build()
    if world > 1:
        dist.barrier()
    mac.lib()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    wl = W.by_name(a.config, a.n)                     # seeded, synthetic; identical on every rank (replicas)
    nu = wl.nu_pre + wl.nu_post
    P = mac.MacProjector(mac.desc_from_workload(wl, smoother=a.smoother, host_staging=0 if a.no_e2e else 3, timing=1), device=dev)
    dv = mac.to_device(wl, dev)
    pristine = [dv[k].clone() for k in ("u", "v", "w")]
    phi = torch.empty(wl.rho.shape, dtype=torch.float64, device=dev)

    def restore():
        for t, p in zip((dv["u"], dv["v"], dv["w"]), pristine):
            t.copy_(p)

    def step():
        rc, st = P.project(dv["beta0"], dv["rho0"], dv["rho"], dv["u"], dv["v"], dv["w"], dv["S"], phi)
        if rc != 0:
            raise RuntimeError(f"maestro_mac_project returned {rc}")
        return st

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()          # runs through warm-up and the timed region; "under load" samples are kept
    for _ in range(max(a.warmup, 0)):
        restore()
        step()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(a.steps)]
    stats = []
    barrier()
    t_wall0 = time.perf_counter()
    for k in range(a.steps):
        restore()                                   # untimed: gives every step its own unprojected U_edge
        ev[k][0].record()
        stats.append(step())
        ev[k][1].record()
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop() if rank == 0 else None
    ms = [e0.elapsed_time(e1) for e0, e1 in ev]
    t_dev = sum(ms) / 1e3
    cycles = stats[-1]["cycles"]
    units_per_rank = sum(wl.ncells * nu * s["cycles"] for s in stats)
    value, t_dev_max = aggregate_replicas(units_per_rank, t_dev, world, dev)
    launches = sum(s["gpu_launches"] for s in stats)

    # roofline of the dominant kernel (level-0 smoother), live from the timed steps
    sm_ms = sum(s["ms_smooth0"] for s in stats)
    sm_n = sum(s["smooth0_timed"] for s in stats)
    peak, peak_src = hbm_peak()
    kname = {0: "k_rbgs_t2", 1: "k_rbgs_color(x2)", 2: "k_rbgs_fused", 3: "k_rbgs_tma", 4: "k_rbgs_tma"}[a.smoother]
    roof = None
    if sm_n > 0 and sm_ms > 0:
        per_launch_ms = sm_ms / sm_n
        sweeps = sum(s["smooth0_sweeps_timed"] for s in stats) / sm_n      # 2 with the two-sweep kernel
        # algorithmic bytes per launch = 48 B per cell per sweep x the cell-sweeps one launch
        # processes; the two-sweep kernel moves half of that through HBM (temporal blocking), so its fraction of the
        # per-sweep roofline can exceed 1 -- `one_pass_bytes` / `frac_one_pass` state what it must move at least
        # `achieved`: what ONE launch must move -- it reads phi, rhs, ax, ay, az and writes phi once, whatever the number
        # of sweeps it applies: 48 B per cell per launch.  This is the physically bounded figure
        # (<= the copy peak).  `per_sweep_*`: SURVEY.md Sec. 8(d)'s unit, 48 B per cell per SWEEP, x the sweeps of a
        # launch; for the two-sweep kernel it can exceed the peak because temporal blocking halves the HBM traffic.
        one_pass = SMOOTHER_BYTES_PER_CELL * wl.ncells
        ach = one_pass / (per_launch_ms * 1e-3) / 1e9
        per_sweep = SMOOTHER_BYTES_PER_CELL * wl.ncells * sweeps / (per_launch_ms * 1e-3) / 1e9
        traffic = ncu_traffic(kname, a.n)
        roof = {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "traffic": traffic, "traffic_source": "ncu --set full capture of this kernel, profiles/roofline_traffic.md (offline, not a live counter)",
                "kernel": kname + " level 0",
                "algorithmic_bytes_per_launch": one_pass, "sweeps_per_launch": sweeps,
                "avg_launch_ms": per_launch_ms, "launches_timed": sm_n, "peak_source": peak_src,
                "frac_of_8000_nominal": ach / 8000.0,
                "dram_traffic_gbs": (traffic / (per_launch_ms * 1e-3) / 1e9) if traffic else None,
                "per_sweep_achieved": per_sweep, "per_sweep_frac": per_sweep / peak, "per_sweep_frac_of_8000_nominal": per_sweep / 8000.0,
                "limiter": "see profiles/ (ncu): shared-memory pipe and fp64 dependency latency at 12 warps per SM (register-bound occupancy), not DRAM; the chip runs at its 1000 W power cap",
                "share_of_step": sm_ms / (t_dev * 1e3) if t_dev > 0 else None}

    # end to end through the host-buffer entry point
    e2e = None
    if not a.no_e2e:
        pin = lambda x: None if x is None else torch.from_numpy(x.copy()).pin_memory()
        hb = {k: pin(getattr(wl, k)) for k in ("beta0", "rho0", "rho", "S", "u", "v", "w")}
        h0 = [torch.from_numpy(getattr(wl, k)) for k in ("u", "v", "w")]
        h2d = sum(hb[k].numel() * 8 for k in hb if hb[k] is not None)
        d2h = sum(hb[k].numel() * 8 for k in ("u", "v", "w"))
        n_e2e = a.steps
        # (i) the single call (maestro_mac_project_host): upload, project, download, one after the other
        single_ms = None
        for k in range(2):                          # one warm-up, one timed
            for t, p in zip((hb["u"], hb["v"], hb["w"]), h0):
                t.copy_(p)
            barrier()
            t0 = time.perf_counter()
            rc, st = P.project_host(hb["beta0"], hb["rho0"], hb["rho"], hb["u"], hb["v"], hb["w"], hb["S"], None)
            torch.cuda.synchronize()
            single_ms = 1e3 * (time.perf_counter() - t0)
            if rc != 0:
                raise RuntimeError(f"maestro_mac_project_host returned {rc}")
        # (ii) the sequence call (maestro_mac_project_host_seq, config 5's pattern): K steps in ONE call; every step's
        # u, v, w go host -> device and come back inside the timed region, overlapped with the neighbouring steps'
        # projections; rho, S and the profiles go up once per call (their bytes are spread over the K steps below)
        for t, p in zip((hb["u"], hb["v"], hb["w"]), h0):
            t.copy_(p)
        outs = [[torch.empty_like(hb[k]).pin_memory() for k in ("u", "v", "w")] for _ in range(3)]
        uvw = 3 * [None]
        for q, key in enumerate(("u", "v", "w")):
            uvw[q] = ([hb[key]] * n_e2e, [outs[k % 3][q] for k in range(n_e2e)])
        e_t, e_units = 0.0, 0
        for rep_ in range(2):                       # a one-step warm-up call, then the timed call of K steps
            K = 1 if rep_ == 0 else n_e2e
            barrier()
            t0 = time.perf_counter()
            rc, sts = P.project_host_seq(hb["beta0"], hb["rho0"], hb["rho"], hb["S"], uvw[0][0][:K], uvw[1][0][:K], uvw[2][0][:K],
                                         uvw[0][1][:K], uvw[1][1][:K], uvw[2][1][:K])
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            if rc != 0:
                raise RuntimeError(f"maestro_mac_project_host_seq returned {rc}")
            if rep_ == 1:
                e_t = dt
                e_units = sum(wl.ncells * nu * st["cycles"] for st in sts)
        once = sum(hb[k].numel() * 8 for k in ("beta0", "rho0", "rho", "S") if hb[k] is not None)
        h2d = d2h + once // n_e2e
        emax = torch.tensor([e_t], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(emax, op=dist.ReduceOp.MAX)
        e2e = {"value": world * e_units / float(emax.item()), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "ms_per_step": 1e3 * float(emax.item()) / n_e2e,
               "api": "maestro_mac_project_host_seq: K steps in one call, pinned host buffers, every step's u, v, w copied in and "
                      "out inside the timed region (overlapped with the neighbouring steps); rho, S, beta0, rho0 once per call",
               "steps_in_call": n_e2e, "h2d_bytes_once_per_call": once,
               "single_call_ms": single_ms, "single_call_api": "maestro_mac_project_host (nothing overlapped; all inputs sent)"}
        del outs
    P.close()
    del dv, pristine, phi
    torch.cuda.empty_cache()

    # the latency-bound configs of BASELINE.json, a few milliseconds each (parity-test cases, not the bench line)
    others = []
    if rank == 0 and world == 1 and not a.no_other_configs:
        for cfg, n_o in (("1", 32), ("2", 128), ("3N", 256)):
            wo = W.by_name(cfg, n_o)
            Po = mac.MacProjector(mac.desc_from_workload(wo), device=dev)
            do = mac.to_device(wo, dev)
            keep = [do[k].clone() for k in ("u", "v", "w")]
            tms, st_o = [], None
            for it in range(3 + 10):
                for t, p in zip((do["u"], do["v"], do["w"]), keep):
                    t.copy_(p)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                rc, st_o = Po.project(do["beta0"], do["rho0"], do["rho"], do["u"], do["v"], do["w"], do["S"], None)
                e1.record()
                torch.cuda.synchronize()
                if rc != 0:
                    raise RuntimeError(f"config {cfg}: maestro_mac_project returned {rc}")
                if it >= 3:
                    tms.append(e0.elapsed_time(e1))
            others.append({"config": cfg, "n": n_o, "ms_per_projection": statistics.median(tms), "cycles": st_o["cycles"],
                           "launches": st_o["gpu_launches"], "timing": "median of 10 after 3 warm-ups, CUDA events"})
            Po.close()
            del do, keep, wo
        torch.cuda.empty_cache()
        # the end-of-step (nodal) projection of SURVEY.md Sec. 8(f) rank 3 on the 256^3 star (cell-centred velocities)
        import numpy as _np
        wo = W.by_name("3N", 256)
        Po = mac.MacProjector(mac.desc_from_workload(wo, nodal=1), device=dev)
        do = mac.to_device(wo, dev)
        cc = [torch.from_numpy(_np.ascontiguousarray(x)).to(dev) for x in W.cell_centred(wo)]
        tms, st_o = [], None
        for it in range(2 + 5):
            uc, vc, wc = (c.clone() for c in cc)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            rc, st_o = Po.nodal_project(do["beta0"], do["rho0"], do["rho"], uc, vc, wc, do["S"], None)
            e1.record()
            torch.cuda.synchronize()
            if rc != 0:
                raise RuntimeError(f"nodal projection returned {rc}")
            if it >= 2:
                tms.append(e0.elapsed_time(e1))
        others.append({"config": "3N, end-of-step nodal projection (maestro_mac_nodal_project)", "n": 256,
                       "ms_per_projection": statistics.median(tms), "cycles": st_o["cycles"], "launches": st_o["gpu_launches"],
                       "timing": "median of 5 after 2 warm-ups, CUDA events"})
        Po.close()
        del do, cc, wo
        torch.cuda.empty_cache()

    cpu = None
    if rank == 0 and world == 1 and not a.no_cpu_baseline:
        # the oracle as it stands on the SAME inputs (one whole projection, all host cores) when the host has the
        # memory (about 15 GB at 512^3, a minute on 16 cores), else on the 256^3 instance of the workload; plus a
        # one-thread figure on a bounded sample (SURVEY.md Sec. 8(d) asks for both)
        ns = a.cpu_sample_n or (a.n if host_mem_available_gb() > 18.0 * (a.n / 512.0) ** 3 + 8.0 else min(256, a.n))
        same = ns == a.n
        dt, cyc, cells, threads, nu_o = cpu_oracle_run(a.config, ns, wl=wl if same else None)
        n1 = min(128, a.n)
        dt1, cyc1, cells1, _, nu1 = cpu_oracle_run(a.config, n1, threads=1)
        cpu = {"value": cells * nu_o * cyc / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": (f"the whole workload: {a.config} at {ns}^3, the same inputs, one full projection, " if same else
                          f"{a.config} at {ns}^3 (same recipe as the {a.n}^3 workload), one full projection, ")
                         + f"{cyc} cycles, {dt:.1f} s",
               "same_config": same, "seconds": dt, "cycles": cyc,
               "one_thread": {"value": cells1 * nu1 * cyc1 / dt1, "unit": UNIT, "cores": 1,
                              "sample": f"{a.config} at {n1}^3, one full projection, {cyc1} cycles, {dt1:.1f} s"},
               "nproc": os.cpu_count(), "cpu_model": cpu_model()}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": a.steps, "warmup": a.warmup,
            "ms_per_step": 1e3 * t_dev_max / max(a.steps, 1), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_label(a.config, a.n), "cells": wl.ncells, "cycles_per_solve": cycles,
                       "levels": stats[-1]["levels"], "smoother": {0: "fused red+black, two sweeps per HBM pass (temporal blocking), TMA-staged", 1: "two-pass reference", 2: "fused single pass, cp.async-staged", 3: "fused single pass, TMA 32x16 tile", 4: "fused red+black, one sweep per pass, TMA-staged"}[a.smoother],
                       "parallelism": "replicas only" if world > 1 else "single GPU",
                       "l2": "inputs larger than L2 (every level-0 array is %.2f GB)" % (wl.ncells * 8 / 1e9)
                             if wl.ncells * 8 > 126e6 else "level arrays fit in L2; no flush (the solve re-reads them by design)",
                       "timing": "CUDA events per step on the call's stream, summed; U_edge restored outside the event pairs"},
            "solves_per_s": world * a.steps / t_dev_max,
            "vcycles_per_s": world * sum(s["cycles"] for s in stats) / t_dev_max,
            "ms_vcycles_per_solve": statistics.mean(s["ms_vcycles"] for s in stats),
            "ms_setup_kernels_per_solve": statistics.mean(s["ms_setup_kernels"] for s in stats),
            "ms_correct_per_solve": statistics.mean(s["ms_correct"] for s in stats),
            "final_rel_residual": stats[-1]["res_history"][-1] if stats[-1]["res_history"] else None,
            "wall_s_timed_region": t_wall,
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roof, "cpu_baseline": cpu,
            "other_configs": others,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    args = parse_args()
    sys.exit(run_reference(args) if args.impl == "reference" else run_ours(args))
