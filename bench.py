#!/usr/bin/env python
"""bench.py -- particle-steps/s of the libm3dk hot path on synthetic tokamak workloads (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A "step" is one pass of the whole hot path over all markers of the workload: field evaluation + slow-manifold Boris
push + delta-f weight (rows a1-a10 of DESIGN.md section 1) and the marker sort by element (row a11) at the configured
interval.  Default workload: BASELINE.json configs[3] (RSAE, 2^24 markers, 256x256 mesh), the configuration the metric
is quoted on ("16M markers on one B200").  Markers shard across ranks with no exchange, so N GPUs
run N shards of the same size: weak scaling, no data-path collective.

Prints ONE JSON line (rank 0).  --impl reference times the CPU oracle (oracle/) on a bounded sample instead.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "particle-steps/sec (fp64 push+field eval+delta-f weight)"
UNIT = "particle-steps/s"
HBM_FALLBACK_GBS = 6650.0           # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # 148 SMs x 64 DFMA lanes x 2 flop x clocks.max.sm


# ---- algorithmic work per marker-step (DESIGN.md section 7 derives these) ---------------------------------------------
def algorithmic_flops(n_modes: int, mode: int = 0) -> float:
    """fp64 operations per marker-step counted from the kernel's formulas: FMA = 2, add / mul = 1,
    reciprocal / rsqrt / sqrt = 1 each (their Newton steps are not counted); minimal-multiplication Horner: value of a
    21-term quintic = 20 FMA, value + d/dxi + d/deta = 38 FMA.  The fp32 arithmetic of the element search is not counted."""
    eq = 2 * (38 + 38 + 20 + 20)              # psi0 and |B|0 with gradients, F0, kappa
    common = 11 + 4 + 68 + 6 + 7              # cylindrical map + local coordinates, scaling, B / E-dagger / Boris, drift, R of x_{l+1}
    if n_modes == 0:
        return eq + common
    pert = 2 * (10 * 20 + 2 * 38)             # E_R E_phi E_Z B_R B_Z (re, im) values; B_par (re, im) value + gradient
    fold = 25 + 25 + 23                       # phase exp(i(n phi - omega t)) for n = 3, folding 5 + 1 complex fields into dw/dt
    weight = 86 + 2                           # coefficients of dw/dt (Eqs. 8-13 incl. kappa_E), w update
    if mode == 1:                             # non-linear trajectories: + B_phi (re, im), total fields, (1 - w)
        return eq + common + weight + 30 + n_modes * (pert + 2 * 2 * 20 + fold + 5)
    if mode == 3:                             # non-linear trajectories in the gyro-averaged fields: mode 1 + the ring of mode 2
        return eq + common + weight + 30 + 60 + 4 * (11 + 4 + 30 + n_modes * (pert + 2 * 2 * 20 + fold)) + 30
    if mode == 2:                             # FLR: ring geometry, then 4 x (map, local coordinates, all 14 polynomials, rotation)
        return eq + common + weight + 60 + 4 * (11 + 4 + 30 + n_modes * (pert + 2 * 2 * 20 + fold)) + 30
    return eq + common + weight + n_modes * (pert + fold)


def algorithmic_bytes_push(n_modes: int, ordered: bool = True) -> float:
    """HBM bytes per marker per push-kernel pass.  Ordered pipeline: 64 B record read + 8 B order
    entry read, 64 B record + 4 B key + 4 B rank written.  SoA path (sort_interval 0): 8 fp64 read, 7 written (mu is
    read-only; w only with modes), element key read + written.  Coefficient tiles are counted as on-chip (shared by the
    markers of an element; about 13 B per marker-step at config 3 if every tile is fetched once per step)."""
    if ordered:
        return 64 + 8 + 64 + 4 + 4
    return 64 + (56 if n_modes else 48) + 4 + 4


def algorithmic_bytes_sort() -> float:
    """Per marker per re-ordering (scan, work-item cut, order list): key + rank + order entry read, order entry written."""
    return 4 + 4 + 8 + 8


# ---- helpers -----------------------------------------------------------------------------------------------------------
def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", float(d.get("sm_max_mhz", 1965.0))
    return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)", 1965.0


TRAFFIC_CSV = os.path.join(ROOT, "profiles", "push_traffic.csv")


def ncu_traffic(config: int, sort_interval: int, mode: int = 0):
    """dram__bytes_read.sum + dram__bytes_write.sum of the push kernels, per push, from the committed ncu --set full
    capture of this workload: profiles/push_traffic.csv, written by `bench.py --traffic-from <ncu raw csv>` together with
    the commit the capture was taken at.  Returns (bytes, commit) or (None, None) when no capture of this configuration
    is recorded."""
    if not os.path.exists(TRAFFIC_CSV):
        return None, None
    found = (None, None)
    with open(TRAFFIC_CSV) as fh:
        for line in fh:
            cols = [c.strip() for c in line.split(",")]
            if len(cols) >= 5 and cols[0] == f"config{config}" and cols[1] == f"si{sort_interval}" and cols[2] == f"mode{mode}":
                found = (float(cols[3]), cols[4])
    return found


def record_traffic(args):
    """--traffic-from: read an `ncu -i <rep> --page raw --csv` export of ONE push (its launches of the push kernels) and
    append its DRAM traffic to profiles/push_traffic.csv with the current commit."""
    import csv
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    with open(args.traffic_from) as fh:
        rows = [r for r in csv.reader(fh) if r]
    hdr, units = rows[0], rows[1]
    kcol = hdr.index("Kernel Name")
    total, kernels = 0.0, []
    for r in rows[2:]:
        if "push_items_kernel" not in r[kcol] and "push_async_kernel" not in r[kcol]:
            continue
        kernels.append(r[kcol].split("(")[0].replace("void ", ""))
        for name in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            c = hdr.index(name)
            total += float(r[c].replace(",", "")) * scale[units[c]]
    if not kernels:
        raise SystemExit("no push kernel in " + args.traffic_from)
    commit = subprocess.run(["git", "-C", ROOT, "rev-parse", "--short", "HEAD"], capture_output=True, text=True).stdout.strip()
    si = 1 if args.sort_interval is None else args.sort_interval
    new_file = not os.path.exists(TRAFFIC_CSV)
    with open(TRAFFIC_CSV, "a") as fh:
        if new_file:
            fh.write("workload,sort_interval,mode,dram_bytes_per_push,commit,date,kernels\n")
        fh.write(f"config{args.config},si{si},mode{args.mode},{total:.0f},{commit or 'unknown'},"
                 f"{time.strftime('%Y-%m-%d')},{'+'.join(kernels)}\n")
    print(f"recorded {total:.0f} B per push ({'+'.join(kernels)}) at {commit}")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for (ts, r) in self.rows if t0 <= ts <= t1 + 0.1] or [r for (_, r) in self.rows[-3:]]
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


ORACLE_MODE = [0]     # set from --mode: the oracle is timed in the same mode as the CUDA path


def oracle_bounded_sample(w, n_sample: int, target_s: float = 15.0):
    """The oracle on a bounded sample sized for about target_s seconds of CPU work on this box: a short calibration run
    (every 1024-th marker, 20 steps) fixes the number of steps for the id = 0 (mod stride) sub-sample."""
    stride = max(1, w.n_markers // n_sample)
    rate, n, secs, cores = oracle_sample_rate(w, max(stride, min(1024, w.n_markers // 1024 or 1)), 20)
    n_s = len(range(0, w.n_markers, stride))
    steps = int(min(6000, max(20, target_s * rate / n_s)))
    return oracle_sample_rate(w, stride, steps) + (stride, steps)


def oracle_sample_rate(w, sample_stride: int, nsteps: int, nthreads: int = 0):
    """The oracle as it stands, FE back-end, OpenMP over markers, on the id = 0 (mod stride) sub-sample."""
    import oracle
    idx = slice(0, None, sample_stride)
    mk = {k: np.ascontiguousarray(v[idx]) for k, v in w.markers.items()}
    mesh, sp = oracle.Mesh.of(w), oracle.species_of(w, mode=ORACLE_MODE[0])
    oracle.push_fe(mesh, sp, {k: v[:256] for k, v in mk.items()}, 1, w.dt)      # touch code and tables
    t0 = time.perf_counter()
    oracle.push_fe(mesh, sp, mk, nsteps, w.dt, nthreads=nthreads)
    dt = time.perf_counter() - t0
    n = mk["x"].shape[0]
    return n * nsteps / dt, n, dt, oracle.max_threads() if nthreads == 0 else nthreads


def build_workload(args, rank: int, tables: bool = True):
    import synth
    from paper_2107_13663_b200 import shard
    # every rank draws its own shard (seed offset by rank): independent markers.  Only rank 0 fits
    # the field tables; the other ranks receive the packed field image from it
    return synth.make_config(args.config, n_markers=args.n_markers, nx=args.nx, dt_gyro=args.dt_gyro,
                             seed=shard.shard_seed(args.config, rank), tables=tables)


def config_dict(args, w, sort_interval, world):
    return {"workload": f"BASELINE.json configs[{args.config}] ({w.name})", "n_markers_per_gpu": w.n_markers,
            "mesh": f"{w.nx}x{w.nx} cells, {w.n_elems} triangles", "n_modes": w.n_modes, "dt": w.dt,
            "sort_interval": sort_interval, "mode": ("linear delta-f", "non-linear trajectories", "linear delta-f + FLR 4-point average",
                     "non-linear trajectories + FLR 4-point average")[args.mode],
            "parallelism": (f"{world} independent marker shard(s), no collective in the push" +
                            ("; field image broadcast from rank 0 (NCCL)" if world > 1 else "")),
            "l2": "inputs larger than L2 (marker state %.0f MB + tables %.0f MB per GPU)" % (
                w.n_markers * 64 / 1e6, (w.eq_coef.nbytes + w.pert_coef.nbytes) / 1e6)}


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle, as it stands, on the box's host cores, on a bounded sample of the workload."""
    if rank != 0:
        return
    w = build_workload(args, 0)
    stride = max(1, w.n_markers // args.ref_sample)
    for _ in range(max(0, min(args.warmup, 1))):
        oracle_sample_rate(w, stride * 8, 1)
    rate, n, secs, cores = oracle_sample_rate(w, stride, args.steps)
    line = {"impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": secs / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(args, w, 0, world),
            "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{n} markers (every {stride}-th of the workload) x {args.steps} steps, {secs:.1f} s"},
            "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    import paper_2107_13663_b200 as m3dk

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libm3dk has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    from paper_2107_13663_b200 import shard
    if rank == 0:
        m3dk.build_all()                 # one rank compiles (if the library is stale); the others wait and load it
    if world > 1:
        dist.barrier()
    w = build_workload(args, rank, tables=(rank == 0))
    # decision D-c: workloads that sort at all run the ordered pipeline, which orders every step
    si = (1 if w.sort_interval > 0 else 0) if args.sort_interval is None else args.sort_interval
    N, K, W = w.n_markers, args.steps, args.warmup

    p = m3dk.Pusher(device=local_rank, verify=False)
    if rank == 0:
        p.fields_create(w.node_RZ, w.tri, w.eq_coef, w.n_tor if w.n_modes else None, w.omega if w.n_modes else None,
                        w.pert_coef if w.n_modes else None)
    if world > 1:
        shard.broadcast_fields(p, dist, w.n_elems, w.n_modes, src=0)
    p.particles_init(w.markers, w.charge, w.mass, w.f0)
    p.set_options(sort_interval=si, mode=args.mode, t0=0.0)
    p.set_push_variant(args.push_variant)
    if args.mode in (2, 3) and si > 0:
        p.set_flr_workspace(nonlinear=(args.mode == 3))           # ring stream of the ordered FLR modes

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- device-resident leg: W warm-up steps, then exactly K timed steps ---------------------------------------
    p.push(W, w.dt)
    p.set_profiling(True)
    sampler = ClockSampler(local_rank) if rank == 0 else None
    time.sleep(0.3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    wall0 = time.time()
    e0.record(p.stream)
    p.push(K, w.dt)
    e1.record(p.stream)
    barrier()
    wall1 = time.time()
    ms = e0.elapsed_time(e1)
    tm = p.timing()
    st = p.stats()
    clocks = sampler.stop(wall0, wall1) if sampler else None
    p.set_profiling(False)

    # ---- end-to-end leg: host buffers through the C ABI (m3dk_push_host), copies inside the timed region ------------------
    # One call = upload + K steps + download of all markers, pipelined by marker chunk.  A chunk is a range of the host
    # buffers and stays that set of markers from call to call.  Markers stream around their flux surface, so a chunk that
    # starts as a range of elements is spread over the whole mesh after some twenty steps (a quarter of the markers per
    # element: the work items fill badly); a chunk that is a radial shell stays a shell and keeps its markers per element.
    if args.e2e_order == "shell":
        # caller's marker order: by minor radius of the loaded position, so that a chunk is a radial shell
        Rm = np.hypot(w.markers["x"], w.markers["y"])
        perm = np.argsort(w.eq.rtheta(Rm, w.markers["z"])[0], kind="stable")
    else:
        perm = np.arange(N)
    host = {k: torch.from_numpy(np.ascontiguousarray(w.markers[k][perm])).pin_memory() for k in m3dk.STATE_KEYS}
    Ke, C_e2e = K, args.e2e_chunks
    if args.e2e_order == "element":
        p.push_host(host, 1, w.dt, n_chunks=1)
    p.push_host(host, 1, w.dt, n_chunks=C_e2e)
    p.set_options(sort_interval=si, mode=args.mode, t0=0.0)
    barrier()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record(p.stream)
    p.push_host(host, Ke, w.dt, n_chunks=C_e2e)
    f1.record(p.stream)
    barrier()
    ms_e2e = f0.elapsed_time(f1)

    ms, ms_e2e = shard.max_over_ranks([ms, ms_e2e], dist if world > 1 else None, device=dev)
    dep = None
    if args.deposit or args.gc:
        # the e2e leg left the device arrays chunk by chunk; the rows below are timed on the state a device-resident
        # push leaves (all markers in the element order of the step before)
        p.push(2, w.dt)
        barrier()
    if args.deposit:
        # row (f)-4 with its exchange step: every rank deposits its shard, the moment tables are summed over the ranks
        need = p.deposit_bytes()
        rhs = torch.empty(need // 8, dtype=torch.float64, device=dev)
        if args.deposit_flags & 2:
            p.set_flr_workspace()       # ordered ring stream of the 4-point deposition
        p.deposit_into(rhs, args.deposit_flags, 0.0)
        shard.allreduce_moments(rhs, dist if world > 1 else None)
        barrier()
        d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        d0.record(p.stream)
        for _ in range(5):
            p.deposit_into(rhs, args.deposit_flags, 0.0)
            shard.allreduce_moments(rhs, dist if world > 1 else None)
        d1.record(p.stream)
        barrier()
        dms, = shard.max_over_ranks([d0.elapsed_time(d1) / 5], dist if world > 1 else None, device=dev)
        dep = (dms, need)
    if rank != 0:
        return

    hbm_gbs, hbm_src, _ = measured_peaks()
    fp64_meas = p.fp64_peak_tflops()
    flops = algorithmic_flops(w.n_modes, args.mode) * N
    bytes_push = algorithmic_bytes_push(w.n_modes, ordered=si > 0) * N
    push_ms = tm["push_ms"] / max(1, tm["push_launches"])
    t_alu, t_hbm = flops / (FP64_NOMINAL_TFLOPS * 1e12), bytes_push / (hbm_gbs * 1e9)
    if t_alu >= t_hbm:
        roof = {"bound": "alu", "achieved": flops / (push_ms * 1e-3) / 1e12, "peak": FP64_NOMINAL_TFLOPS,
                "unit": "TFLOP/s", "peak_source": "nominal fp64: 148 SM x 64 DFMA/clk x 2 x 1.965 GHz (DESIGN.md 7)"}
    else:
        roof = {"bound": "hbm", "achieved": bytes_push / (push_ms * 1e-3) / 1e9, "peak": hbm_gbs, "unit": "GB/s",
                "peak_source": hbm_src}
    roof["frac"] = roof["achieved"] / roof["peak"]
    traffic, traffic_commit = ncu_traffic(args.config, si, args.mode)
    if roof["bound"] == "alu":
        # the measured FP64 peak (register-resident DFMA chains, m3dk_fp64_peak_tflops) beside the nominal one
        roof["frac_of_measured_peak"] = roof["achieved"] / fp64_meas if fp64_meas > 0 else None
    roof.update({"kernel": "push kernel (a1-a10)", "launch_ms": push_ms, "launches": tm["push_launches"],
                 "share_of_step": tm["push_ms"] / ms, "traffic": traffic, "traffic_commit": traffic_commit,
                 "fp64_peak_measured_tflops": fp64_meas,
                 "flops_per_marker_step": algorithmic_flops(w.n_modes, args.mode),
                 "hbm_bytes_per_marker_step": algorithmic_bytes_push(w.n_modes, ordered=si > 0),
                 "sort_ms_per_sort": tm["sort_ms"] / max(1, tm["sort_launches"]), "sorts": tm["sort_launches"]})
    # whole-step roofline: the binding one of (all flops / fp64 peak) and (all HBM bytes incl. sorts / HBM bandwidth)
    step_bytes = bytes_push + algorithmic_bytes_sort() * N * tm["sort_launches"] / K
    t_bind = max(t_alu, step_bytes / (hbm_gbs * 1e9))
    roof["step_frac_of_binding_roofline"] = t_bind / (ms / K * 1e-3)

    line = {"metric": METRIC, "value": shard.whole_job_rate([N] * world, K, ms), "unit": UNIT, "n_gpus": world, "steps": K,
            "warmup": W, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": config_dict(args, w, si, world),
            "clocks": clocks, "gpu_launches": tm["kernel_launches"],
            "e2e": {"value": shard.whole_job_rate([N] * world, Ke, ms_e2e), "unit": UNIT, "h2d_bytes_per_step": 64 * N / Ke,
                    "d2h_bytes_per_step": 64 * N / Ke,
                    "note": f"m3dk_push_host: one upload + {Ke} steps + one download per call (PAPER.md:237), pipelined in "
                            f"{C_e2e if C_e2e else 'an automatic number of'} marker chunks; host buffers pinned, order of the markers: {args.e2e_order}"},
            "roofline": roof, "n_lost": st["n_lost"]}
    if args.gc:
        # row (f)-3: RK4 guiding-centre steps on the same markers (x, y, z as X; v_par = 0.5 for every marker)
        vpar = torch.full((N,), 0.5, dtype=torch.float64, device=dev)
        p.gc_push_into(3, w.dt, vpar)
        torch.cuda.synchronize(dev)
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record(p.stream)
        p.gc_push_into(10, w.dt, vpar)
        g1.record(p.stream)
        torch.cuda.synchronize(dev)
        gms = g0.elapsed_time(g1) / 10
        line["gc"] = {"ms_per_step": gms, "particle_steps_per_s": N / (gms * 1e-3),
                      "fields": "equilibrium + perturbation (reading G26)" if args.mode in (1, 3) and w.n_modes else "equilibrium",
                      "note": "m3dk_gc_push, RK4 on Eqs. (1)-(4) (SURVEY.md 8(f)-3); 4 field evaluations per step"}
    if dep is not None:
        dms, need = dep
        dbytes = (68.0 * N + need)            # 8 fp64 + element key per marker read, the table cleared and accumulated
        line["deposit"] = {"ms": dms, "markers_per_s": N * world / (dms * 1e-3), "table_bytes": need,
                           "hbm_bytes": dbytes, "hbm_frac": dbytes / (dms * 1e-3) / (hbm_gbs * 1e9),
                           "flags": args.deposit_flags,
                           "note": "m3dk_deposit (flags: 1 = B1par term of Eq. 16, 2 = 4-point FLR, 4 = d = w + B1par/B*par), "
                                   "delta-function shape (SURVEY.md 8(f)-4)" +
                                   (f", then NCCL all-reduce of the {need} B table over {world} ranks" if world > 1 else "")}
    if world == 1 and not args.no_cpu_baseline:
        rate, n, secs, cores, stride, rsteps = oracle_bounded_sample(w, args.ref_sample)
        line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"{n} markers (every {stride}-th of the workload) x {rsteps} steps, {secs:.1f} s"}
    print(json.dumps(line), flush=True)


def run_sweep(args):
    """BASELINE.json configs[4]: marker count x dt x ordering interval on the config-3 equilibrium and perturbation; one
    JSON line per point (particle-steps/s and the fraction of the binding roofline), single GPU, device-resident timing.
    Not the driver's contract line: a table generator for BASELINE.md."""
    import torch
    import synth
    import paper_2107_13663_b200 as m3dk

    torch.cuda.set_device(0)
    m3dk.build_all()
    hbm_gbs, _, _ = measured_peaks()
    K, W = args.steps, args.warmup
    for n in args.sweep_n:
        for dtg in args.sweep_dt:
            w = synth.make_config(4, n_markers=n, dt_gyro=dtg)
            for si in args.sweep_si:
                p = m3dk.Pusher(device=0, verify=False)
                p.fields_create(w.node_RZ, w.tri, w.eq_coef, w.n_tor, w.omega, w.pert_coef)
                p.particles_init(w.markers, w.charge, w.mass, w.f0)
                p.set_options(sort_interval=si, t0=0.0)
                p.push(W, w.dt)
                p.set_profiling(True)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                e0.record(p.stream)
                p.push(K, w.dt)
                e1.record(p.stream)
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1) / K
                tm = p.timing()
                t_alu = algorithmic_flops(w.n_modes) * n / (FP64_NOMINAL_TFLOPS * 1e12)
                t_hbm = (algorithmic_bytes_push(w.n_modes, ordered=si > 0) + algorithmic_bytes_sort() * tm["sort_launches"] / K) * n / (hbm_gbs * 1e9)
                row = {"sweep_point": {"n_markers": n, "dt_gyro": dtg, "sort_interval": si},
                       "value": n / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms,
                       "push_ms": tm["push_ms"] / max(1, tm["push_launches"]),
                       "binding": "alu" if t_alu >= t_hbm else "hbm",
                       "frac_of_binding_roofline": max(t_alu, t_hbm) / (ms * 1e-3),
                       "n_lost": p.stats()["n_lost"]}
                print(json.dumps(row), flush=True)
                if args.sweep_out:
                    new_file = not os.path.exists(args.sweep_out)
                    with open(args.sweep_out, "a") as fh:
                        if new_file:
                            fh.write("n_markers,dt_gyro,sort_interval,particle_steps_per_s,ms_per_step,push_ms,binding,"
                                     "frac_of_binding_roofline,n_lost,steps,warmup\n")
                        fh.write(f"{n},{dtg},{si},{row['value']:.6e},{ms:.5f},{row['push_ms']:.5f},{row['binding']},"
                                 f"{row['frac_of_binding_roofline']:.4f},{row['n_lost']},{K},{W}\n")
                p.close()
                del p
                torch.cuda.empty_cache()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--n-markers", type=int, default=None)
    ap.add_argument("--nx", type=int, default=None)
    ap.add_argument("--dt-gyro", type=float, default=None)
    ap.add_argument("--sort-interval", type=int, default=None)
    ap.add_argument("--ref-sample", type=int, default=65536, help="markers in the oracle's bounded sample")
    ap.add_argument("--mode", type=int, default=0, choices=[0, 1, 2, 3],
                    help="0: linear delta-f (the headline); 1: non-linear trajectories (SURVEY.md 8(f)-1); "
                         "2: linear delta-f with the 4-point gyro-average (8(f)-2)")
    ap.add_argument("--gc", action="store_true", help="also time m3dk_gc_push (SURVEY.md 8(f)-3) on the final state")
    ap.add_argument("--deposit", action="store_true", help="also time m3dk_deposit (SURVEY.md 8(f)-4) on the final state")
    ap.add_argument("--deposit-flags", type=int, default=1, help="flags of the timed m3dk_deposit (1 B1par, 2 FLR, 4 Bstar)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-order", choices=("shell", "element", "loaded"), default="shell",
                    help="order of the host buffers of the e2e leg: radial shells, the element order a one-chunk call returns, as loaded")
    ap.add_argument("--e2e-chunks", type=int, default=0, help="marker chunks of the pipelined host-buffer call (e2e leg); 0 = the library chooses")
    ap.add_argument("--push-variant", type=int, default=0, choices=[0, 1],
                    help="m3dk_set_push_variant: 0 = default kernel, 1 = asynchronously staged kernel (A/B comparison)")
    ap.add_argument("--traffic-from", default=None,
                    help="record the DRAM traffic of the push kernels from an `ncu --page raw --csv` export into "
                         "profiles/push_traffic.csv (with the current commit) and exit")
    ap.add_argument("--sweep", action="store_true", help="configs[4] sweep: one JSON line per (n, dt, sort interval)")
    ap.add_argument("--sweep-out", default=None, help="append one CSV row per sweep point to this file")
    ap.add_argument("--sweep-n", type=int, nargs="+", default=[1 << 20, 1 << 22, 1 << 24, 1 << 26])
    ap.add_argument("--sweep-dt", type=float, nargs="+", default=[1.0, 4.0, 16.0])
    ap.add_argument("--sweep-si", type=int, nargs="+", default=[1, 10, 0])
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    ORACLE_MODE[0] = args.mode
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.traffic_from:
        record_traffic(args)
        return
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if args.sweep:
        if rank == 0:
            run_sweep(args)
        return
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=__import__("torch").device("cuda", local_rank))
    try:
        run_ours(args, rank, world, local_rank)
    finally:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
