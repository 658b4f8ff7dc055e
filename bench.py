#!/usr/bin/env python
"""bench.py -- grid points/s of twojmax=10 fp64 bispectrum descriptors (BASELINE.json metric) on one B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--twojmax 10] [--shard none|z] [--impl native|reference]

A step = one pass of the whole hot path (tile binning -> compute_ui -> compute_zi/compute_bi -> writer)
over the full grid of the workload (default: config 2, 256-atom solid Al on a 90^3 grid, the configuration the metric
is quoted on).  `value` is measured through mala_bispectrum_grid with the output resident in HBM; `e2e` through
mala_bispectrum_grid_host with a pinned HOST output (the device->host copy of all ncomp x npoints doubles is inside the
timed region).  N > 1: one process per GPU (spawned here through torch.distributed.run when the launcher has not done
it), no collective on the data path: `--shard none` = independent replicas of the whole grid
(weak scaling), `--shard z` = ONE grid split into z-slabs balanced by non-empty points (strong scaling).
`--impl reference` times the CPU oracle (oracle/) as it stands on the host cores -- the only baseline that exists.
Other workloads: --config 200cube | binary, --twojmax 2..14.
"""
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

METRIC = "grid points/s of twojmax=10 fp64 bispectrum descriptors; % of B200 FP64 peak"
UNIT = "points/s"
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # 148 SMs x 64 DFMA/clk/SM x 2 flop x 1.965 GHz = 37.2


def flop_model(twojmax):
    """Algorithmic flops: what the method must compute using the standard
    half-column symmetry -- not instruction counts.  Counted here from the index ranges themselves; at twojmax = 10:
    235 recursion steps, 271 U elements, 3,444 Z elements, 61,332 product terms, 13,230 outer steps, i.e.
    F_pair = 5,844, F_Z = 666,240, F_B = 13,958."""
    tj = int(twojmax)
    triples = [(j1, j2, j) for j1 in range(tj + 1) for j2 in range(j1 + 1) for j in range(j1 - j2, min(tj, j1 + j2) + 1, 2) if j >= j1]
    nelem = sum((J + 1) * (J // 2 + 1) for J in range(tj + 1))
    steps = sum((J + 1) * (J // 2 + 1) for J in range(1, tj + 1)) - sum(J + 1 for J in range(2, tj + 1, 2))
    nz = terms = outer = 0
    for J1, J2, J in triples:
        sh = (J1 + J2 - J) // 2
        for mb in range(J // 2 + 1):
            mid = (J % 2 == 0) and (mb == J // 2)
            nb = min(J1, mb + sh) - max(0, mb + sh - J2) + 1
            for ma in range((J // 2 if mid else J) + 1):
                na = min(J1, ma + sh) - max(0, ma + sh - J2) + 1
                nz += 1
                terms += na * nb
                outer += nb
    return {"ncomp": len(triples), "nelem": nelem, "F_PAIR": 20 * steps + 4 * nelem + 60, "F_Z": 10 * terms + 4 * outer,
            "F_B": 4 * nz + 2 * len(triples), "terms": terms}


def ncu_traffic(workload_key, kernel, live_ms):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed `ncu --set full` capture
    (profiles/traffic.json, written from the capture named there).  Returned only when that capture's kernel duration
    agrees with the duration measured live in this run within 3 % -- otherwise the capture is stale and the answer is None."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            table = json.load(f)
    except (OSError, ValueError):
        return None, "no profiles/traffic.json"
    ent = table.get(f"{workload_key}:{kernel}")
    if not ent:
        return None, "no capture for this workload/kernel"
    if live_ms <= 0 or abs(ent["ncu_ms"] - live_ms) > 0.03 * live_ms:
        return None, f"capture {ent['source']} is stale: {ent['ncu_ms']:.2f} ms under ncu vs {live_ms:.2f} ms live"
    return float(ent["dram_bytes"]), ent["source"]


def parse_args():
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=5)
    p.add_argument("--warmup", type=int, default=3)
    p.add_argument("--config", default="2", choices=["1", "2", "3", "4", "5", "200cube", "binary"],
                   help="1-5: BASELINE.json configs; 200cube: config 2's atoms on the paper's 200^3 grid; binary: two species")
    p.add_argument("--twojmax", type=int, default=None, help="override the workload's twojmax (default 10)")
    p.add_argument("--shard", default="none", choices=["none", "z"],
                   help="N > 1: none = every rank computes the whole grid (replicas), z = one grid split into z-slabs")
    p.add_argument("--impl", default="native", choices=["native", "reference"])
    p.add_argument("--descriptor", default="bispectrum", choices=["bispectrum", "gaussian"],
                   help="gaussian: the SURVEY 8(f) f2 path (mala_gaussian_grid), a separate metric line")
    p.add_argument("--sigma", type=float, default=0.5, help="Gaussian width for --descriptor gaussian")
    p.add_argument("--ldos", action="store_true",
                   help="SURVEY 8(f) f1: descriptors + the descriptor->LDOS network in one call (mala_bispectrum_ldos_grid), a separate metric line")
    p.add_argument("--force", action="store_true",
                   help="SURVEY 8(f) f3: the adjoint of the descriptor map (mala_bispectrum_force_adjoint), a separate metric line")
    p.add_argument("--zi-impl", type=int, default=0,
                   help="compute_zi kernel: 0 automatic, 1 table-driven, 2 per-triple (twojmax 10), 3 anti-diagonal, 4 register-tiled blocks")
    p.add_argument("--yi-impl", type=int, default=0, help="compute_yi kernel of --force: 0 automatic (2), 1 table-driven, 2 block kernel with Y in fixed point, 3 block kernel with fp64 atomics")
    p.add_argument("--ui-impl", type=int, default=0,
                   help="compute_ui kernel: 0 automatic, 1 column, 2 sampling (twojmax 1..10), 3 pipelined sampling (twojmax 8..14)")
    p.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg (profiling runs)")
    p.add_argument("--no-e2e", action="store_true", help="skip the host-output leg (profiling runs)")
    args = p.parse_args()
    args.config = int(args.config) if args.config.isdigit() else args.config
    return args


# ---------------------------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md "clocks line")
# ---------------------------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.rows = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.gpu)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); smax.append(float(f[2])); power.append(float(f[3]))
            except ValueError:
                continue
            for name, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": float(max(power))}


# ---------------------------------------------------------------------------------------------------------------
# workload facts used by the flop model
# ---------------------------------------------------------------------------------------------------------------
def workload_counts(w):
    """(pairs, non-empty points) of the whole grid.  Periodic bulk systems: every point has neighbors and the mean
    neighbor count of a uniform grid is exactly rho * 4/3 pi rcut^3.  The non-periodic cluster is counted directly."""
    if all(w.pbc):
        vol = abs(np.linalg.det(w.box))
        nbar = sum(int((w.types == t).sum()) / vol * 4.0 / 3.0 * np.pi * (2.0 * w.rcutfac * r) ** 3 for t, r in enumerate(w.radelem))
        return nbar * w.npoints, w.npoints
    rcut = 2.0 * w.rcutfac * w.radelem[0]
    nx, ny, nz = w.ngrid
    fx, fy, fz = np.arange(nx) / nx, np.arange(ny) / ny, np.arange(nz) / nz
    cnt = np.zeros((nz, ny, nx), dtype=np.int32)
    ax = fx[None, None, :, None] * w.box[0] + fy[None, :, None, None] * w.box[1]
    for z0 in range(0, nz, 8):
        pts = ax + fz[z0:z0 + 8, None, None, None] * w.box[2] + np.asarray(w.origin)
        for a in w.pos:
            cnt[z0:z0 + 8] += (((pts - a) ** 2).sum(-1) < rcut * rcut)
    return float(cnt.sum()), int((cnt > 0).sum())


def plane_costs(w):
    """relative cost of every z-plane for the slab partition of --shard z: non-empty points (exact for the cluster in
    vacuum, uniform for periodic bulk)"""
    nx, ny, nz = w.ngrid
    if all(w.pbc):
        return [1.0] * nz
    rcut = 2.0 * w.rcutfac * max(w.radelem)
    fx, fy, fz = np.arange(nx) / nx, np.arange(ny) / ny, np.arange(nz) / nz
    ax = fx[None, :, None] * w.box[0] + fy[:, None, None] * w.box[1]
    cost = []
    for z in range(nz):
        pts = ax + fz[z] * w.box[2] + np.asarray(w.origin)
        hit = np.zeros((ny, nx), dtype=bool)
        for a in w.pos:
            hit |= ((pts - a) ** 2).sum(-1) < rcut * rcut
        cost.append(float(hit.sum()) + 0.02 * nx * ny)   # empty points still cost their 8 * ncomp bytes of fill
    return cost


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return {"hbm_gbs": d.get("hbm_gbs"), "source": "measured (MEASURED_PEAKS.json)", "sm_max_mhz": d.get("sm_max_mhz")}
    return {"hbm_gbs": 6650.0, "source": "fallback (B200_PROFILING.md)", "sm_max_mhz": 1965.0}


# ---------------------------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py executes oracle/)
# ---------------------------------------------------------------------------------------------------------------
def oracle_rate(w, seconds, seed=7):
    """points/s of the oracle, as it stands, on a seeded random sample of the grid sized to take about `seconds`."""
    import oracle
    rng = np.random.default_rng(seed)
    kw = w.snap_params()
    probe = rng.integers(0, w.npoints, 64 * max(oracle.num_threads(), 1))
    t0 = time.perf_counter()
    oracle.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, sample=probe, **kw)
    dt = time.perf_counter() - t0
    n = int(min(max(probe.size, seconds / max(dt, 1e-6) * probe.size), 400000))
    sample = rng.integers(0, w.npoints, n)
    t0 = time.perf_counter()
    oracle.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, sample=sample, **kw)
    dt = time.perf_counter() - t0
    # per-core rate: one thread on >= 2,000 points (SURVEY.md 8(d) "Oracle timing beside it" (ii)), bounded to ~6 s
    threads = oracle.num_threads()
    n1 = int(min(max(2000, 0.25 * n / max(threads, 1)), 6.0 * (n / dt) / max(threads, 1) + 2000))
    s1 = rng.integers(0, w.npoints, n1)
    oracle.set_num_threads(1)
    t0 = time.perf_counter()
    oracle.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, sample=s1, **kw)
    dt1 = time.perf_counter() - t0
    oracle.set_num_threads(threads)
    return n / dt, n, dt, threads, n1 / dt1, n1


def run_reference(args, w, rank, world):
    """--impl reference: the CPU oracle on the host cores, rank 0 only.  Each step = a bounded seeded sample."""
    if rank != 0:
        return
    import oracle
    rng = np.random.default_rng(11)
    kw = w.snap_params()
    threads = oracle.num_threads()
    # calibrate the per-step sample so the whole run stays near two minutes
    probe = rng.integers(0, w.npoints, 64 * max(threads, 1))
    t0 = time.perf_counter()
    oracle.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, sample=probe, **kw)
    per_pt = (time.perf_counter() - t0) / probe.size
    budget = 100.0 / max(args.steps + args.warmup, 1)
    n = int(min(max(256, budget / per_pt), w.npoints))
    times = []
    for it in range(args.warmup + args.steps):
        sample = rng.integers(0, w.npoints, n)
        t0 = time.perf_counter()
        oracle.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, sample=sample, **kw)
        if it >= args.warmup:
            times.append(time.perf_counter() - t0)
    total = float(sum(times))
    value = n * len(times) / total
    sample_desc = f"{n} seeded random grid points of {w.name} per step (of {w.npoints}); rate is per point, not extrapolated"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(w, "cpu oracle"),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample_desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(w, path, parallelism="replicas"):
    return {"workload": f"config{w.extra.get('cfg', '?')}:{w.name}", "natoms": int(w.pos.shape[0]), "ngrid": list(map(int, w.ngrid)),
            "npoints": int(w.npoints), "twojmax": int(w.twojmax), "ncomp": flop_model(w.twojmax)["ncomp"],
            "rcut": [float(2 * w.rcutfac * r) for r in w.radelem] if len(w.radelem) > 1 else float(2 * w.rcutfac * w.radelem[0]),
            "path": path, "parallelism": parallelism,
            "l2": "no flush: each step streams the U_tot workspace and the output (both far larger than the 126 MB L2)"}


# ---------------------------------------------------------------------------------------------------------------
# multi-rank plumbing (torch.distributed; replicas only -- there is no exchange step on this path)
# ---------------------------------------------------------------------------------------------------------------
def dist_setup(args):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def reduce_max_sum(value_max, value_sum, world, backend_device=None):
    """(max over ranks of value_max, sum over ranks of value_sum).  world == 1: identity."""
    if world == 1:
        return float(value_max), float(value_sum)
    import torch
    import torch.distributed as dist
    dev = backend_device if backend_device is not None else "cpu"
    a = torch.tensor([float(value_max)], dtype=torch.float64, device=dev)
    b = torch.tensor([float(value_sum)], dtype=torch.float64, device=dev)
    dist.all_reduce(a, op=dist.ReduceOp.MAX)
    dist.all_reduce(b, op=dist.ReduceOp.SUM)
    return float(a.item()), float(b.item())


def run_native(args, w, rank, world, local):
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    from paper_2411_19617_b200 import MalaSnap, mala_snap_fp64_peak, slabs

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    fm = flop_model(w.twojmax)
    nt = fm["ncomp"]
    nx, ny, nz = (int(v) for v in w.ngrid)
    sharded = (args.shard == "z" and world > 1)
    z0, z1 = (0, nz)
    if sharded:   # one grid, rank r takes slab r of a partition balanced by non-empty points; atoms replicated, nothing exchanged
        z0, z1 = slabs.weighted_z_slabs(plane_costs(w), world)[rank]
    npts = (z1 - z0) * ny * nx
    snap = MalaSnap(**w.snap_params())
    assert snap.ncomp == nt
    if args.zi_impl:
        snap.set_option("zi_impl", args.zi_impl)
    if args.ui_impl:
        snap.set_option("ui_impl", args.ui_impl)
    stream = torch.cuda.current_stream()
    out = torch.empty((max(npts, 1), nt), dtype=torch.float64, device=dev)
    call = lambda: snap.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, z0, z1, out=out, stream=stream)

    # ---- device-resident leg ------------------------------------------------------------------------------
    snap.set_option("timing", 1)
    for _ in range(args.warmup):
        call()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.15)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    ktimes = []
    launches = 0
    barrier()
    for a, b in evs:
        a.record(stream)
        call()
        b.record(stream)
        ktimes.append(snap.kernel_times())  # waits for this step's kernels; steps are serial on the stream anyway
        launches += snap.last_stats()["kernels"]
    barrier()
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in evs]
    total_ms = float(sum(step_ms))
    total_ms, total_pts = reduce_max_sum(total_ms, npts * args.steps, world, dev)
    value = total_pts / (total_ms * 1e-3)
    stats = snap.last_stats()
    snap.set_option("timing", 0)

    # ---- roofline of the dominant kernel (compute_zi_bi: rows a5 + a6 + a7) --------------------------------
    pairs, nonempty = workload_counts(w)
    if sharded:   # this rank's share (uniform bulk: by points; the cluster: by its plane costs)
        pc = plane_costs(w)
        frac = sum(pc[z0:z1]) / sum(pc)
        pairs, nonempty = pairs * frac, nonempty * frac
    zi_ms = float(np.mean([k["compute_zi_bi"][0] for k in ktimes]))
    zi_launches = ktimes[-1]["compute_zi_bi"][1]
    ui_ms = float(np.mean([k["compute_ui"][0] for k in ktimes]))
    bin_ms = float(np.mean([k["tile_bin"][0] for k in ktimes]))
    zi_flop = nonempty * (fm["F_Z"] + fm["F_B"])           # per step = summed over that step's launches
    achieved = zi_flop / (zi_ms * 1e-3) / 1e12 if zi_ms > 0 else 0.0
    peak_meas, mhz_eff = mala_snap_fp64_peak(stream)
    kernel = snap.zi_kernel_name()
    roofline = {"bound": "alu", "kernel": kernel, "achieved": achieved, "peak": FP64_NOMINAL_TFLOPS,
                "unit": "TFLOP/s", "frac": achieved / FP64_NOMINAL_TFLOPS,
                "peak_source": "nominal FP64 FMA pipe: 148 SM x 64 DFMA/clk x 2 x 1.965 GHz (DESIGN.md 'FP64 roofline')",
                "peak_measured_dfma": peak_meas, "frac_of_measured_dfma": achieved / peak_meas if peak_meas > 0 else None,
                "dfma_probe_sm_mhz": mhz_eff, "traffic": None,
                "flop_per_point": {"pair": fm["F_PAIR"], "zi": fm["F_Z"], "bi": fm["F_B"]},
                "flop_per_launch": zi_flop / max(zi_launches, 1), "launches_per_step": zi_launches, "ms_per_launch": zi_ms / max(zi_launches, 1),
                "kernel_ms_per_step": {"tile_bin": bin_ms, "compute_ui": ui_ms, "compute_zi_bi": zi_ms},
                "compute_ui_tflops": pairs * fm["F_PAIR"] / (ui_ms * 1e-3) / 1e12 if ui_ms > 0 else None,
                "step_model_tflops": (pairs * fm["F_PAIR"] + zi_flop) / (total_ms / args.steps * 1e-3) / 1e12 if world == 1 else None}
    wl_key = f"config{w.extra.get('cfg')}/tj{w.twojmax}"
    roofline["traffic"], roofline["traffic_source"] = ncu_traffic(wl_key, kernel, zi_ms / max(zi_launches, 1))
    peaks = load_peaks()
    roofline["hbm_gbs_step"] = (npts * nt * 8 + 2 * (nonempty / 32) * fm["nelem"] * 32 * 16) / (total_ms / args.steps * 1e-3) / 1e9 if world == 1 else None
    roofline["hbm_peak_gbs"] = peaks["hbm_gbs"]
    roofline["hbm_peak_source"] = peaks["source"]
    # the fill of empty tiles is the HBM-bound part of tile_bin (config 4): 8 * ncomp bytes per empty point
    if nonempty < npts and bin_ms > 0 and not sharded:
        roofline["tile_bin_fill_gbs"] = (npts - nonempty) * nt * 8 / (bin_ms * 1e-3) / 1e9

    # ---- end-to-end leg: host output buffer, D2H inside the timed region ------------------------------------
    e2e = None
    if not args.no_e2e:
        host = torch.empty((max(npts, 1), nt), dtype=torch.float64, pin_memory=True)
        call_host = lambda: snap.bispectrum_grid_host(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, z0, z1, out=host, stream=stream)
        for _ in range(max(1, min(args.warmup, 2))):
            call_host()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            call_host()  # returns after the last device->host copy has completed
        torch.cuda.synchronize()
        e2e_s = time.perf_counter() - t0
        e2e_s, e2e_pts = reduce_max_sum(e2e_s, npts * args.steps, world, dev)
        h2d = int(w.pos.nbytes + w.types.nbytes + 9 * 8 + 3 * 8 + 3 * 4 + 3 * 4)
        e2e = {"value": e2e_pts / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": int(npts * nt * 8),
               "ms_per_step": 1e3 * e2e_s / args.steps,
               "note": "mala_bispectrum_grid_host: HOST atoms in, pinned HOST descriptors out; D2H overlapped with the kernels of the next z-chunk"}
        del host

    # ---- CPU oracle beside it (rank 0, N = 1 only) ---------------------------------------------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        rate, n, dt, threads, rate1, n1 = oracle_rate(w, seconds=12.0)
        cpu = {"value": rate, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": f"{n} seeded random grid points of {w.name} (of {w.npoints}) in {dt:.1f} s wall on {threads} threads",
               "one_thread": {"value": rate1, "unit": UNIT, "sample": f"{n1} seeded random grid points on 1 thread"},
               "cpu_model": cpu_model(), "host_cores_online": os.cpu_count()}

    snap.close()
    if world > 1:
        torch.distributed.destroy_process_group()
    if rank != 0:
        return
    cfg = workload_config(w, "mala_bispectrum_grid (device out)", "z-slab shards of one grid" if sharded else "replicas")
    cfg.update({"chunks_per_step": stats["chunks"], "workspace_bytes": stats["workspace_bytes"], "ghost_atoms": stats["ghosts"]})
    if sharded:
        cfg["rank0_slab"] = [z0, z1]
    line = {"metric": METRIC if w.twojmax == 10 else METRIC.replace("twojmax=10", f"twojmax={w.twojmax}"),
            "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": cfg, "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline, "cpu_baseline": cpu, "pct_of_fp64_peak_step": None}
    if roofline["step_model_tflops"] is not None:
        line["pct_of_fp64_peak_step"] = 100.0 * roofline["step_model_tflops"] / FP64_NOMINAL_TFLOPS
    print(json.dumps(line), flush=True)


def run_gaussian(args, w, rank, world, local):
    """--descriptor gaussian: grid points/s of mala_gaussian_grid (row f2).  Same contract: device leg, e2e leg with a pinned
    host copy of the result, oracle baseline.  Flop model per point: 9 flop per candidate-free distance test is not
    algorithmic, so only the hits count: 8 (distance) + 1 sqrt + 22 (exp) + 2 = 33 flop per neighbor within the cutoff."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        torch.distributed.init_process_group("nccl", device_id=dev)
    from paper_2411_19617_b200 import MalaSnap
    npts, nty = w.npoints, len(w.radelem)
    snap = MalaSnap(**w.snap_params())
    stream = torch.cuda.current_stream()
    out = torch.empty((npts, nty), dtype=torch.float64, device=dev)
    host = torch.empty((npts, nty), dtype=torch.float64, pin_memory=True)
    call = lambda: snap.gaussian_grid(args.sigma, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, out=out, stream=stream)

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    snap.set_option("timing", 1)
    for _ in range(args.warmup):
        call()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.15)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    launches, kms = 0, []
    barrier()
    for a, b in evs:
        a.record(stream)
        call()
        b.record(stream)
        launches += snap.last_stats()["kernels"]
        kms.append(snap.kernel_times())
    barrier()
    clocks = sampler.stop()
    total_ms = float(sum(a.elapsed_time(b) for a, b in evs))
    total_ms, total_pts = reduce_max_sum(total_ms, npts * args.steps, world, dev)
    value = total_pts / (total_ms * 1e-3)
    g_ms = float(np.mean([k["other"][0] for k in kms]))
    bin_ms = float(np.mean([k["tile_bin"][0] for k in kms]))
    pairs, _ = workload_counts(w)
    peaks = load_peaks()
    achieved = pairs * 33 / (g_ms * 1e-3) / 1e12
    roofline = {"bound": "alu", "kernel": "gaussian_grid_kernel", "achieved": achieved, "peak": FP64_NOMINAL_TFLOPS, "unit": "TFLOP/s",
                "frac": achieved / FP64_NOMINAL_TFLOPS, "traffic": None, "flop_per_launch": pairs * 33,
                "kernel_ms_per_step": {"tile_bin": bin_ms, "gaussian_grid": g_ms},
                "hbm_out_gbs": npts * nty * 8 / (g_ms * 1e-3) / 1e9, "hbm_peak_gbs": peaks["hbm_gbs"],
                "note": "neither roofline binds at these sizes: 33 flop per neighbor and 8 B per point leave the kernel latency-bound"}
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        call()
        host.copy_(out, non_blocking=True)
        torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_s, e2e_pts = reduce_max_sum(e2e_s, npts * args.steps, world, dev)
    h2d = int(w.pos.nbytes + w.types.nbytes + 9 * 8 + 3 * 8 + 3 * 4 + 3 * 4)
    e2e = {"value": e2e_pts / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": int(npts * nty * 8),
           "ms_per_step": 1e3 * e2e_s / args.steps}
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        rng = np.random.default_rng(7)
        n = 200000
        sample = rng.integers(0, npts, n)
        pts = oracle.grid_points(w.box, w.origin, w.ngrid, sample=sample)
        t0 = time.perf_counter()
        oracle.gaussian_points(pts, w.pos, w.types, w.box, w.origin, w.pbc, sigma=args.sigma, rcutfac=w.rcutfac, radelem=w.radelem, wj=w.wj)
        dt = time.perf_counter() - t0
        cpu = {"value": n / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"{n} seeded random grid points of {w.name} (of {npts}) in {dt:.1f} s wall"}
    snap.close()
    if world > 1:
        torch.distributed.destroy_process_group()
    if rank != 0:
        return
    cfg = workload_config(w, "mala_gaussian_grid (device out)")
    cfg.update({"ncomp": nty, "sigma": args.sigma})
    line = {"metric": "grid points/s of Gaussian descriptors (SURVEY 8(f) f2)", "value": value, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg, "clocks": clocks,
            "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)


def run_ldos(args, w, rank, world, local):
    """--ldos: grid points/s of mala_bispectrum_ldos_grid (row f1): descriptors, then the 91 -> 256 -> 256 -> 241 network on the
    tensor cores, LDOS (fp32) resident in HBM; e2e adds the device->host copy of the LDOS.  Roofline of the network kernel:
    bound "tensor", 2 * sum_l w_l w_{l+1} flop per grid point against the TF32 peak (measured bf16 burst peak x the nominal
    TF32 : BF16 ratio of 1/2)."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        torch.distributed.init_process_group("nccl", device_id=dev)
    from paper_2411_19617_b200 import MalaMlp, MalaSnap, bispectrum_ldos_grid, workloads

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    fm = flop_model(w.twojmax)
    sizes = (fm["ncomp"], 256, 256, 241)
    ws, bs, shift, scale = workloads.ldos_network(sizes=sizes)
    npts = w.npoints
    snap = MalaSnap(**w.snap_params())
    net = MalaMlp(ws, bs, "leaky_relu", True, shift, scale)
    stream = torch.cuda.current_stream()
    out = torch.empty((npts, sizes[-1]), dtype=torch.float32, device=dev)
    call = lambda: bispectrum_ldos_grid(snap, net, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, out=out, stream=stream)
    snap.set_option("timing", 1)
    for _ in range(args.warmup):
        call()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.15)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    ktimes, launches = [], 0
    barrier()
    for a, b in evs:
        a.record(stream)
        call()
        b.record(stream)
        ktimes.append(snap.kernel_times())
        launches += snap.last_stats()["kernels"]
    barrier()
    clocks = sampler.stop()
    total_ms = float(sum(a.elapsed_time(b) for a, b in evs))
    total_ms, total_pts = reduce_max_sum(total_ms, npts * args.steps, world, dev)
    value = total_pts / (total_ms * 1e-3)
    stats = snap.last_stats()
    mlp_ms = float(np.mean([k["other"][0] for k in ktimes]))
    mlp_launches = ktimes[-1]["other"][1]
    kms = {"tile_bin": float(np.mean([k["tile_bin"][0] for k in ktimes])), "compute_ui": float(np.mean([k["compute_ui"][0] for k in ktimes])),
           "compute_zi_bi": float(np.mean([k["compute_zi_bi"][0] for k in ktimes])), "mlp_forward": mlp_ms}
    flop_pt = 2 * sum(a * b for a, b in zip(sizes[:-1], sizes[1:]))
    rows = 32 * stats["tiles"]                    # the network runs on whole tiles (ragged lanes included)
    achieved = flop_pt * npts / (mlp_ms * 1e-3) / 1e12 if mlp_ms > 0 else 0.0
    bf16 = None
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            bf16 = json.load(f).get("bf16_tflops")
    except (OSError, ValueError):
        pass
    peak_src = "MEASURED_PEAKS.json bf16 burst peak x 0.5 (nominal TF32 : BF16)" if bf16 else "fallback: nominal 2250 x 0.5 (B200_PROFILING.md)"
    peak = 0.5 * (bf16 if bf16 else 2250.0)
    roofline = {"bound": "tensor", "kernel": "mlp_forward_kernel", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "peak_source": peak_src, "traffic": None, "flop_per_point": flop_pt, "flop_per_launch": flop_pt * npts / max(mlp_launches, 1),
                "launches_per_step": mlp_launches, "ms_per_launch": mlp_ms / max(mlp_launches, 1), "kernel_ms_per_step": kms,
                "rows_processed_per_step": rows, "network": list(sizes), "operand_dtype": "tf32 (fp32 accumulate)",
                "note": "the network is ~1.5 % of the step; it is bound by streaming its 0.62 MB of weights from L2 once per 128-row tile, "
                        "not by the tensor pipe (DESIGN.md section 13)"}
    roofline["traffic"], roofline["traffic_source"] = ncu_traffic(f"config{w.extra.get('cfg')}/tj{w.twojmax}", "mlp_forward_kernel",
                                                                  mlp_ms / max(mlp_launches, 1))
    host = torch.empty((npts, sizes[-1]), dtype=torch.float32, pin_memory=True)
    # e2e: the grid in z-slabs of eight planes through the z_begin / z_end arguments of the entry point, the device->host copy
    # of one slab (a second stream) behind the kernels of the next; calls on one handle are serialised by the library
    copy_stream = torch.cuda.Stream(device=dev)
    plane_pts = w.ngrid[0] * w.ngrid[1]
    slabs_z = [(za, min(za + 8, w.ngrid[2])) for za in range(0, w.ngrid[2], 8)]

    def e2e_step():
        for za, zb in slabs_z:
            part = out[za * plane_pts:zb * plane_pts]
            bispectrum_ldos_grid(snap, net, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, za, zb, out=part, stream=stream)
            done = torch.cuda.Event()
            done.record(stream)
            copy_stream.wait_event(done)
            with torch.cuda.stream(copy_stream):
                host[za * plane_pts:zb * plane_pts].copy_(part, non_blocking=True)
        torch.cuda.synchronize()

    e2e_step()   # slab-sized workspaces and the copy stream exist before the clock starts
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()
    e2e_s = time.perf_counter() - t0
    e2e_s, e2e_pts = reduce_max_sum(e2e_s, npts * args.steps, world, dev)
    h2d = int(w.pos.nbytes + w.types.nbytes + 9 * 8 + 3 * 8 + 3 * 4 + 3 * 4)
    e2e = {"value": e2e_pts / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": int(npts * sizes[-1] * 4),
           "ms_per_step": 1e3 * e2e_s / args.steps,
           "note": "mala_bispectrum_ldos_grid per z-slab of eight planes: HOST atoms in, pinned HOST LDOS out; D2H of a slab behind the kernels of the next"}
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        from oracle import mlp_oracle
        rng = np.random.default_rng(7)
        n = 60000
        sample = rng.integers(0, npts, n)
        t0 = time.perf_counter()
        B = oracle.bispectrum_grid(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, sample=sample, **w.snap_params())
        mlp_oracle.mlp_forward(B, ws, bs, "leaky_relu", True, shift, scale)
        dt = time.perf_counter() - t0
        cpu = {"value": n / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"{n} seeded random grid points of {w.name} (of {npts}) in {dt:.1f} s wall: C descriptor oracle + numpy fp64 network"}
    net.close()
    snap.close()
    if world > 1:
        torch.distributed.destroy_process_group()
    if rank != 0:
        return
    cfg = workload_config(w, "mala_bispectrum_ldos_grid (device out)")
    cfg.update({"ncomp_out": sizes[-1], "network": list(sizes), "chunks_per_step": stats["chunks"], "workspace_bytes": stats["workspace_bytes"]})
    line = {"metric": "grid points/s of LDOS vectors: twojmax=%d fp64 bispectrum descriptors + descriptor->LDOS network (SURVEY 8(f) f1)" % w.twojmax,
            "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64 descriptors, tf32 network", "data": "synthetic",
            "config": cfg, "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)


def force_flop_model(twojmax):
    """Algorithmic flops of row f3 per non-empty grid point (compute_yi) and per (grid point, neighbor) pair (compute_dedr),
    counted from the index ranges.  Y^C[ma][mb] over half columns receives, for every bispectrum
    component (j1, j2, j), the Z-type contributions (j1, j2) -> j, (j, j2) -> j1 and (j, j1) -> j2 (the distinct ones: with
    equal entries two or all three coincide and are computed once): 10 flop per
    product term and 4 per outer step, as for compute_zi.  compute_dedr repeats the U recursion of the pair (F_PAIR) and
    dots every coefficient of levels 0 .. twojmax-1 with two Y columns for the four Cayley-Klein derivatives (4 complex
    multiply-adds = 32 flop) plus the weight sum (8 flop per element of U)."""
    tj = int(twojmax)
    fm = flop_model(tj)
    triples = [(j1, j2, j) for j1 in range(tj + 1) for j2 in range(j1 + 1) for j in range(j1 - j2, min(tj, j1 + j2) + 1, 2) if j >= j1]
    terms = outer = 0
    for j1, j2, j in triples:
        for A, B, C in dict.fromkeys(((j1, j2, j), (j, j2, j1), (j, j1, j2))):   # equal entries: the same contraction once
            sh = (A + B - C) // 2
            for mb in range(C // 2 + 1):
                mid = (C % 2 == 0) and (mb == C // 2)
                nb = min(A, mb + sh) - max(0, mb + sh - B) + 1
                for ma in range((C // 2 if mid else C) + 1):
                    na = min(A, ma + sh) - max(0, ma + sh - B) + 1
                    terms += na * nb
                    outer += nb
    nelem_lower = sum((J + 1) * (J // 2 + 1) for J in range(tj))   # coefficients of levels 0 .. tj-1
    return {"F_Y": 10 * terms + 4 * outer, "Y_terms": terms, "F_DEDR_PAIR": fm["F_PAIR"] + 32 * nelem_lower + 8 * fm["nelem"]}


def run_force(args, w, rank, world, local):
    """--force: grid points/s of mala_bispectrum_force_adjoint (row f3, Eqs. (44)-(45) PAPER.md:418-428): beta[point][ncomp]
    resident in HBM -> g[natoms][3].  e2e adds the host->device copy of beta from pinned memory and the device->host read of g."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        torch.distributed.init_process_group("nccl", device_id=dev)
    from paper_2411_19617_b200 import MalaSnap, mala_snap_fp64_peak

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    fm, ffm = flop_model(w.twojmax), force_flop_model(w.twojmax)
    nt, npts, natoms = fm["ncomp"], w.npoints, int(w.pos.shape[0])
    snap = MalaSnap(**w.snap_params())
    stream = torch.cuda.current_stream()
    gen = torch.Generator(device="cpu").manual_seed(7)
    beta_host = torch.randn((npts, nt), dtype=torch.float64, generator=gen).pin_memory()
    beta = beta_host.to(dev)
    g = torch.zeros((natoms, 3), dtype=torch.float64, device=dev)

    def call():
        g.zero_()
        snap.force_adjoint(beta, w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, out=g, stream=stream)

    if args.yi_impl:
        snap.set_option("yi_impl", args.yi_impl)
    snap.set_option("timing", 1)
    for _ in range(args.warmup):
        call()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.15)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    ktimes, launches = [], 0
    barrier()
    for a, b in evs:
        a.record(stream)
        call()
        b.record(stream)
        ktimes.append(snap.kernel_times())
        launches += snap.last_stats()["kernels"]
    barrier()
    clocks = sampler.stop()
    total_ms = float(sum(a.elapsed_time(b) for a, b in evs))
    total_ms, total_pts = reduce_max_sum(total_ms, npts * args.steps, world, dev)
    value = total_pts / (total_ms * 1e-3)
    stats = snap.last_stats()
    kms = {"tile_bin": float(np.mean([k["tile_bin"][0] for k in ktimes])), "compute_ui": float(np.mean([k["compute_ui"][0] for k in ktimes])),
           "compute_yi": float(np.mean([k["compute_zi_bi"][0] for k in ktimes])), "compute_dedr": float(np.mean([k["other"][0] for k in ktimes]))}
    pairs, nonempty = workload_counts(w)
    yi_launches = ktimes[-1]["compute_zi_bi"][1]
    yi_flop = nonempty * ffm["F_Y"]
    achieved = yi_flop / (kms["compute_yi"] * 1e-3) / 1e12 if kms["compute_yi"] > 0 else 0.0
    peak_meas, mhz_eff = mala_snap_fp64_peak(stream)
    step_flop = yi_flop + pairs * (fm["F_PAIR"] + ffm["F_DEDR_PAIR"])
    roofline = {"bound": "alu", "kernel": "compute_yi_fix_kernel" if args.yi_impl in (0, 2) else "compute_yi_block_kernel", "achieved": achieved, "peak": FP64_NOMINAL_TFLOPS, "unit": "TFLOP/s",
                "frac": achieved / FP64_NOMINAL_TFLOPS,
                "peak_source": "nominal FP64 FMA pipe: 148 SM x 64 DFMA/clk x 2 x 1.965 GHz (DESIGN.md 'FP64 roofline')",
                "peak_measured_dfma": peak_meas, "frac_of_measured_dfma": achieved / peak_meas if peak_meas > 0 else None, "traffic": None,
                "flop_per_point": {"yi": ffm["F_Y"], "dedr_per_pair": ffm["F_DEDR_PAIR"], "ui_per_pair": fm["F_PAIR"]},
                "flop_per_launch": yi_flop / max(yi_launches, 1), "launches_per_step": yi_launches,
                "ms_per_launch": kms["compute_yi"] / max(yi_launches, 1), "kernel_ms_per_step": kms,
                "compute_dedr_tflops": pairs * ffm["F_DEDR_PAIR"] / (kms["compute_dedr"] * 1e-3) / 1e12 if kms["compute_dedr"] > 0 else None,
                "step_model_tflops": step_flop / (total_ms / args.steps * 1e-3) / 1e12 if world == 1 else None}
    roofline["traffic"], roofline["traffic_source"] = ncu_traffic(f"config{w.extra.get('cfg')}/tj{w.twojmax}", roofline["kernel"],
                                                                  kms["compute_yi"] / max(yi_launches, 1))
    # end to end: beta from pinned host memory, g back to the host, every step
    g_host = torch.empty((natoms, 3), dtype=torch.float64, pin_memory=True)
    # the grid in z-slabs through z_begin / z_end (the call adds each slab's contribution to g): the host->device copy of the
    # next slab's beta (a second stream) runs behind the kernels of the current one
    copy_stream = torch.cuda.Stream(device=dev)
    plane_pts = w.ngrid[0] * w.ngrid[1]
    slabs_z = [(za, min(za + 16, w.ngrid[2])) for za in range(0, w.ngrid[2], 16)]

    def e2e_step():
        g.zero_()
        copied = []
        for za, zb in slabs_z:     # every copy is enqueued up front; the compute stream waits slab by slab
            with torch.cuda.stream(copy_stream):
                beta[za * plane_pts:zb * plane_pts].copy_(beta_host[za * plane_pts:zb * plane_pts], non_blocking=True)
                ev = torch.cuda.Event()
                ev.record(copy_stream)
            copied.append(ev)
        for (za, zb), ev in zip(slabs_z, copied):
            stream.wait_event(ev)
            snap.force_adjoint(beta[za * plane_pts:zb * plane_pts], w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, za, zb, out=g, stream=stream)
        g_host.copy_(g, non_blocking=True)
        torch.cuda.synchronize()

    copy_stream.wait_stream(stream)
    e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()
    e2e_s = time.perf_counter() - t0
    e2e_s, e2e_pts = reduce_max_sum(e2e_s, npts * args.steps, world, dev)
    h2d = int(beta_host.numel() * 8 + w.pos.nbytes + w.types.nbytes + 9 * 8 + 3 * 8 + 3 * 4 + 3 * 4)
    e2e = {"value": e2e_pts / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": int(natoms * 3 * 8),
           "ms_per_step": 1e3 * e2e_s / args.steps,
           "note": "mala_bispectrum_force_adjoint per z-slab of 16 planes: pinned HOST beta in (H2D of the next slab behind the kernels), HOST g out"}
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        rng = np.random.default_rng(7)
        n = 256 * max(oracle.num_threads(), 1)
        sample = rng.integers(0, npts, n)
        pts = oracle.grid_points(w.box, w.origin, w.ngrid, sample=sample)
        b = rng.normal(size=(n, nt))
        t0 = time.perf_counter()
        oracle.bispectrum_grad_points(pts, w.pos, w.types, w.box, w.origin, w.pbc, beta=b, want_dB=False, **w.snap_params())
        dt = time.perf_counter() - t0
        cpu = {"value": n / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"{n} seeded random grid points of {w.name} (of {npts}) in {dt:.1f} s wall: forward-mode dB/dR of the C oracle"}
    snap.close()
    if world > 1:
        torch.distributed.destroy_process_group()
    if rank != 0:
        return
    cfg = workload_config(w, "mala_bispectrum_force_adjoint (beta and g resident in HBM)")
    cfg.update({"chunks_per_step": stats["chunks"], "workspace_bytes": stats["workspace_bytes"]})
    line = {"metric": "grid points/s of the descriptor adjoint g = sum beta dB/dR (SURVEY 8(f) f3), twojmax=%d fp64" % w.twojmax,
            "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)


def spawn_ranks(args):
    """`python bench.py --gpus N` without a launcher: start the N ranks ourselves, exactly as the driver would
    (torch.distributed.run, one process per GPU, rendezvous on 127.0.0.1), and pass their output through."""
    import socket
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    args = parse_args()
    rank, world, local = dist_setup(args)
    if world != args.gpus and world > 1:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}")
    if args.gpus > 1 and world == 1:
        if args.impl == "reference":
            args.gpus = 1    # the oracle arm runs on rank 0 alone
        else:
            raise SystemExit(spawn_ranks(args))
    from paper_2411_19617_b200 import workloads
    w = workloads.make(args.config, twojmax=args.twojmax)
    w.extra["cfg"] = args.config
    if args.impl == "reference":
        run_reference(args, w, rank, world)
        return
    if args.descriptor == "gaussian":
        run_gaussian(args, w, rank, world, local)
        return
    if args.ldos:
        run_ldos(args, w, rank, world, local)
        return
    if args.force:
        run_force(args, w, rank, world, local)
        return
    run_native(args, w, rank, world, local)


if __name__ == "__main__":
    main()
