#!/usr/bin/env python
"""bench.py -- throughput of the channel-flow hot path on B200 (metric: BASELINE.json).

A "step" is one pass of the whole hot path over one synthetic field: chan_run over one step with snapshot and
statistics cadence 1 = the plane statistics (a14) and the filtered database of the entry state (a13) fused into one full RK3 step
(3 substeps = rows a1-a12 of DESIGN.md).  ``value`` counts only the 3 substeps' grid points (Mpoint*RK-substeps/s), so the
filter and statistics time is inside the denominator but earns no credit; ``substep_only`` gives the
rate of the substeps alone.  Inputs are resident in HBM before the timed region; ``e2e`` repeats the
measurement through the *_host entry points with pinned host buffers (state in, state + filtered
database + statistics out, every step).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3|cfg4|cfg5|mid|cfg1] [--impl reference]

N > 1 (torchrun): the path does not shard without an exchange step, so ranks run
independent replicas; value = all ranks' points / max-over-ranks time; scaling "weak".
``--impl reference`` times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "Mpoint*RK-substeps/s fp64"
UNIT = "Mpoint*substeps/s"

# Compulsory HBM traffic of each kernel class in bytes per grid point it processes (
# one complex field pass = 8 B/point).  The SURVEY groups are the section 8(d) figures.
BYTES_PER_POINT = {
    "d1_forward": 16, "derive_down": 48, "derive_up": 40, "zfft_inv": 120, "xfft_prod": 108, "zfft_fwd": 60,
    "y1": 56, "y2": 80, "y3": 88, "y4": 72, "stats": 48, "transpose": 16,   # y1..y4 = sweeps SA..SD, derive_* = SE, SF
    "planes_merged": 288,     # K2 + K3 + K4 of neighbouring chunks in one launch (120 + 108 + 60)
}
SURVEY_GROUPS = {
    "K2 z-pad + inverse z-FFT": (["zfft_inv"], 120),
    "K3 x-FFT . products . x-FFT": (["xfft_prod"], 108),
    "K4 forward z-FFT + truncate": (["zfft_fwd"], 60),
    "K5+K1 y-phase": (["y1", "y2", "y3", "y4", "y5", "d1_forward", "derive_down", "derive_up", "mean"], 144),
    "K2+K3+K4 plane phase": (["zfft_inv", "xfft_prod", "zfft_fwd", "planes_merged"], 288),
}


# Per-launch hardware counters of the hot kernels come from the committed `ncu --set full` table of THIS round
# (profiles/r2_summary.md names the command): roofline.traffic = dram__bytes_read.sum + dram__bytes_write.sum, and the
# shared-memory roof uses l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.  They are not measured live (a number taken
# under a profiler is never a bench value): the JSON says which file and row they come from, and they are null when
# the table has no launch of the same kernel with the same grid.
NCU_TABLE = os.path.join("profiles", "r2_ncu_full_cfg5slab.csv")
KERNEL_OF_CLASS = {"xfft_prod": "k_xfft_prod_s<3", "xfft_prod_filter": "k_xfft_prod_s<7", "zfft_inv": "k_zfft_inv_s", "zfft_fwd": "k_zfft_fwd_s",
                   "planes_merged": "k_planes_s", "y1": "k_sa(", "y2": "k_sb(", "y3": "k_sc(", "y4": "k_sd(", "derive_down": "k_se(",
                   "derive_up": "k_sf(", "stats": "k_stats("}
FP64_PEAK_DERIVED_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12     # 148 SMs x 64 fp64 FMA/clk x 2 x 1965 MHz (guide's unit counts): a note beside the measured peak
SMEM_BYTES_PER_CLK_PER_SM = 128                              # one 128-byte shared-memory wavefront per clock per SM


def ncu_row(cls, grid):
    """Row of the committed ncu table for kernel class `cls` launched with `grid` (tuple), or None."""
    import csv
    path = os.path.join(ROOT, NCU_TABLE)
    name = KERNEL_OF_CLASS.get(cls)
    if not name or not os.path.exists(path):
        return None
    with open(path, newline="") as fh:
        rows = list(csv.DictReader(fh))
    want = "(" + ", ".join(str(int(g)) for g in grid) + ")"
    for r in rows:
        if name in (r.get("Kernel Name") or "") and (r.get("Grid Size") or "").replace(" ", "") == want.replace(" ", ""):
            return r
    return None


def xpass_flops_per_point(nx, nz):
    """"5 N log2 N" flops of the x pass (a4-a6) per grid point: five packed complex transforms of length 3nx/2 plus the
    products on each of the 3nz/2 rows of a plane."""
    import math
    mx, mz = 3 * nx // 2, 3 * nz // 2
    return mz * (5 * 5.0 * mx * math.log2(mx) + 15.0 * mx) / (nx * nz)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p))["hbm_gbs"], "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons while the timed region runs (B200_PROFILING.md clocks line)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.stop = index, [], threading.Event()
        self.t = threading.Thread(target=self.run, daemon=True)

    def run(self):
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self.stop.wait(0.2)

    def __enter__(self):
        self.t.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.t.join(timeout=6)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        sm = [float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(len(r) > 3 + k and r[3 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": float(self.rows[0][1]), "samples": len(self.rows),
                "power_w_max": max(float(r[2]) for r in self.rows), "reasons": reasons}


def max_over_ranks(ms, world, device):
    """Device-timed milliseconds of this rank -> the maximum over all ranks (the job's time).  `device` is where the
    backend wants its tensors (cuda for NCCL, cpu for gloo in the CPU tests)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(npts, substeps, world, ms_max):
    """Whole-job Mpoint*substeps/s of `world` replicas that each advanced npts points by `substeps` substeps."""
    return world * npts * substeps / (ms_max * 1e-3) / 1e6


def pick_workload(name, free_bytes):
    from paper_1808_06461_b200 import inputs
    if name != "auto":
        return name
    for cand in ("cfg5", "cfg4", "cfg3"):
        c = inputs.CONFIGS[cand]
        F = c["nx"] * c["ny"] * c["nz"] * 8
        if 10.3 * F + 8e9 < free_bytes:      # workspace (10 fields + plane chunks) + filter output + slack
            return cand
    return "mid"


def oracle_sample(cfg_name, steps, warmup):
    """The oracle as it stands on a bounded sample: same ny, mesh, Re, dt, box resolution; nx x nz cut down."""
    from oracle.channel import ChannelOracle
    from paper_1808_06461_b200 import inputs
    c = inputs.config(cfg_name)
    snx, snz = min(c["nx"], 48), min(c["nz"], 32)
    cs = inputs.config(cfg_name, nx=snx, nz=snz, lx=c["lx"] * snx / c["nx"], lz=c["lz"] * snz / c["nz"],
                       cut=(min(c["cut"][0], snx // 2 - 1), min(c["cut"][1], snz // 2 - 1)))
    v, phi, omy = (t.numpy() for t in inputs.fluctuations(cs))
    o = ChannelOracle(cs["nx"], cs["ny"], cs["nz"], cs["lx"], cs["lz"], cs["y"], cs["re"], cs["dt"])
    o.set_state(v, phi, omy, cs["U"], cs["W"])
    pts = cs["nx"] * cs["ny"] * cs["nz"]

    def one():
        o.step()
        o.filter_store(*cs["cut"])
        o.stats_accumulate()

    for _ in range(warmup):
        one()
    t0 = time.perf_counter()
    for _ in range(steps):
        one()
    dt = time.perf_counter() - t0
    sample = (f"oracle.ChannelOracle, {steps} x (step + filter_store + stats) on a {snx}x{cs['ny']}x{snz} sub-box of {cfg_name} "
              f"(same mesh, Re, dt, dx, dz; {pts} points)")
    return 3 * pts * steps / dt / 1e6, dt / steps * 1e3, sample


def _oracle_worker(cfg_name, barrier, q):
    """One process of the all-core baseline: builds its oracle, waits for the others, runs one sample step."""
    import numpy  # noqa: F401  (spawned: fresh interpreter)
    os.environ.setdefault("OMP_NUM_THREADS", "1")
    from oracle.channel import ChannelOracle
    from paper_1808_06461_b200 import inputs
    c = inputs.config(cfg_name)
    snx, snz = min(c["nx"], 48), min(c["nz"], 32)
    cs = inputs.config(cfg_name, nx=snx, nz=snz, lx=c["lx"] * snx / c["nx"], lz=c["lz"] * snz / c["nz"],
                       cut=(min(c["cut"][0], snx // 2 - 1), min(c["cut"][1], snz // 2 - 1)))
    v, phi, omy = (t.numpy() for t in inputs.fluctuations(cs))
    o = ChannelOracle(cs["nx"], cs["ny"], cs["nz"], cs["lx"], cs["lz"], cs["y"], cs["re"], cs["dt"])
    o.set_state(v, phi, omy, cs["U"], cs["W"])
    barrier.wait(timeout=600)
    t0 = time.perf_counter()
    o.step()
    o.filter_store(*cs["cut"])
    o.stats_accumulate()
    q.put((cs["nx"] * cs["ny"] * cs["nz"], t0, time.perf_counter()))


def oracle_all_cores(cfg_name, ncores):
    """The oracle as it stands on every host core at once: one independent sub-box per core (the oracle itself is
    single-threaded numpy; the wall-normal stages are independent per mode, so a slab of modes per core is how it
    would be spread), all started together; value = all points x 3 substeps / (last finish - first start)."""
    import multiprocessing as mp
    ctx = mp.get_context("spawn")
    bar, q = ctx.Barrier(ncores), ctx.Queue()
    procs = [ctx.Process(target=_oracle_worker, args=(cfg_name, bar, q)) for _ in range(ncores)]
    for p in procs:
        p.start()
    res = [q.get(timeout=700) for _ in procs]
    for p in procs:
        p.join(timeout=60)
    wall = max(r[2] for r in res) - min(r[1] for r in res)
    pts = sum(r[0] for r in res)
    return 3 * pts / wall / 1e6, (f"{ncores} processes x (step + filter_store + stats) of oracle.ChannelOracle, one 48 x ny x 32 sub-box of "
                                  f"{cfg_name} each, started together; {pts} points in {wall:.1f} s")


def cufft_reference_line(c, dev, npl=8):
    """Context only (north_star: "cuFFT may be timed only as a reference line, not used in the product"): the same plane
    transforms of one substep -- 6 fields spectral -> physical with 3/2 padding, 3 fields back with truncation -- through
    torch.fft (cuFFT, complex128) on a chunk of `npl` planes, scaled to the ny planes of the workload.  No products."""
    import torch
    nx, nz, ny = c["nx"], c["nz"], c["ny"]
    nxh, mx, mz = nx // 2, 3 * nx // 2, 3 * nz // 2
    g = torch.Generator(device=dev).manual_seed(1)
    x = torch.view_as_complex(torch.randn((npl, nz, nxh, 2), generator=g, dtype=torch.float64, device=dev))
    pad = torch.zeros((npl, mz, mx // 2 + 1), dtype=torch.complex128, device=dev)

    def inverse(f):
        pad.zero_()
        pad[:, : nz // 2, :nxh] = f[:, : nz // 2]
        pad[:, mz - (nz // 2 - 1):, :nxh] = f[:, nz // 2 + 1:]
        return torch.fft.irfft(torch.fft.ifft(pad, dim=1), n=mx, dim=2)

    def forward(r):
        s = torch.fft.fft(torch.fft.rfft(r, dim=2)[:, :, :nxh], dim=1)
        return torch.cat([s[:, : nz // 2], s[:, :1] * 0, s[:, mz - (nz // 2 - 1):]], dim=1)

    for _ in range(3):
        ph = inverse(x)
        forward(ph)
    e = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    torch.cuda.synchronize(dev)
    e[0].record()
    for _ in range(6):
        ph = inverse(x)
    e[1].record()
    for _ in range(3):
        forward(ph)
    e[2].record()
    for _ in range(6):      # the two inverse transforms alone, no padding copies
        torch.fft.irfft(torch.fft.ifft(pad[:, :, :nxh], dim=1), n=mx, dim=2)
    e[3].record()
    torch.cuda.synchronize(dev)
    k = ny / npl
    return {"what": "torch.fft (cuFFT) complex128, same padded plane transforms of one substep, products excluded",
            "ms_per_substep": (e[0].elapsed_time(e[1]) + e[1].elapsed_time(e[2])) * k,
            "inverse_6_fields_ms": e[0].elapsed_time(e[1]) * k, "forward_3_fields_ms": e[1].elapsed_time(e[2]) * k,
            "inverse_transforms_alone_ms": e[2].elapsed_time(e[3]) * k, "planes_timed": npl}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = args.workload
    if wl == "auto":        # the workload the GPU arm picks on this box (cfg5 on a 180 GB B200)
        wl = "cfg5"
        try:
            import torch
            if torch.cuda.is_available():
                wl = pick_workload("auto", torch.cuda.mem_get_info(0)[0])
        except Exception:
            pass
    steps = max(1, min(args.steps, 3))
    val1, ms1, sample1 = oracle_sample(wl, steps, min(args.warmup, 1))
    ncores = len(os.sched_getaffinity(0))
    val, ms, sample, cores = val1, ms1, sample1, 1
    if ncores > 1:
        try:                                  # the oracle as it stands on every host core: one sub-box per core
            val, sample = oracle_all_cores(wl, ncores)
            cores = ncores
            c = __import__("paper_1808_06461_b200.inputs", fromlist=["x"]).config(wl)
            pts = ncores * min(c["nx"], 48) * c["ny"] * min(c["nz"], 32)
            ms = 3 * pts / (val * 1e6) * 1e3
        except Exception:
            val, ms, sample, cores = val1, ms1, sample1, 1
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps if cores == 1 else 1,
            "warmup": min(args.warmup, 1), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": {"workload": wl, "note": "CPU oracle on a bounded sample"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "single_core": {"value": val1, "unit": UNIT, "cores": 1, "sample": sample1}},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--workload", default="auto")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cufft-line", action="store_true")
    ap.add_argument("--tuning", default="", help="chan_tuning_t overrides, e.g. plane_overlap=1,maxradix_x=16 (experiments)")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` on its own: become N ranks, one per GPU, exactly as the driver launches them
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
                                  "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:])
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    import __graft_entry__ as entry
    entry.build()
    from paper_1808_06461_b200 import binding, inputs

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    W = max(args.warmup, 3)
    K = max(args.steps, 1)

    free_b, total_b = torch.cuda.mem_get_info(dev)
    wl = pick_workload(args.workload, free_b)
    c = inputs.config(wl)
    npts = c["nx"] * c["ny"] * c["nz"]
    F = npts * 8
    kxc, kzc = c["cut"]

    # ---- inputs: built slab by slab on the device into pinned host buffers (they are also the e2e leg's host
    # side), handed to the library once through chan_set_state_host, so that the state is resident in HBM
    # inside the library's workspace before the timed region and no second device copy competes for memory
    shape = (c["nz"], c["nx"] // 2, c["ny"])
    try:
        hv, hp, ho = (torch.empty(shape, dtype=torch.complex128, pin_memory=True) for _ in range(3))
        pinned = True
    except RuntimeError:
        hv, hp, ho = (torch.empty(shape, dtype=torch.complex128) for _ in range(3))
        pinned = False
    inputs.fluctuations(c, device=dev, zchunk=max(1, min(c["nz"], (1 << 31) // (c["nx"] // 2 * c["ny"] * 16))), out=(hv, hp, ho))
    hU = torch.from_numpy(c["U"]).clone()
    hW = torch.from_numpy(c["W"]).clone()
    torch.cuda.empty_cache()
    tuning = {k: int(v_) for k, v_ in (kv.split("=") for kv in args.tuning.split(",") if kv)}
    ch = binding.Channel(c["nx"], c["ny"], c["nz"], c["lx"], c["lz"], c["y"], c["re"], c["dt"], tuning=tuning or None)
    plan_text, tune = ch.debug_describe(), ch.debug_get_tuning()
    merged = tune["plane_overlap"] == 2
    ws_bytes = ch.workspace_bytes()
    ch.bind(dev)
    ch.set_state_host(hv, hp, ho, hU, hW)
    fout = torch.empty((10, c["ny"], 2 * kzc + 1, kxc + 1), dtype=torch.complex128, device=dev)
    stream = ch.stream
    fring = fout.unsqueeze(0)            # a ring of one slot over the same memory

    def one_step():
        # statistics and filtered database of the state the step starts from, then the step: chan_step_filter forms the
        # filter products from the z-padded planes of the first substep (no inverse z sweep of its own)
        # (chan_run with every = 1: the statistics come out of the (0,0) modes of the fp64 database it writes, L124)
        ch.run(1, 1, 1, kxc, kzc, ring=fring)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(W):
        one_step()
    barrier()
    l0 = ch.debug_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ch.debug_profile(True)
    with ClockSampler(local) as clk:
        barrier()
        e0.record(stream)
        for _ in range(K):
            one_step()
        e1.record(stream)
        barrier()
    ch.debug_profile(False)
    ms_total = e0.elapsed_time(e1)
    prof = ch.debug_profile_read()
    launches = ch.debug_launch_count() - l0
    ms_total_max = max_over_ranks(ms_total, world, dev)
    value = job_value(npts, 3 * K, world, ms_total_max)
    # finite-state check: a blown-up field would make the timing meaningless (the ten filtered variables
    # are linear and quadratic in every velocity and vorticity component)
    finite = bool(torch.isfinite(torch.view_as_real(fout)).all().item())

    # ---- substeps alone -----------------------------------------------------------------------------
    barrier()
    e0.record(stream)
    for _ in range(K):
        ch.step()
    e1.record(stream)
    barrier()
    ms_sub = e0.elapsed_time(e1)
    substep_only = {"value": 3 * npts * K / (ms_sub * 1e-3) / 1e6, "unit": UNIT, "ms_per_substep": ms_sub / (3 * K)}

    # ---- roofline of the dominant kernel + SURVEY groups ---------------------------------------------
    peak, peak_src = measured_peaks()
    sub_classes = {k: v_ for k, v_ in prof.items() if v_[1] > 0}
    dom = max((k for k in sub_classes if k in BYTES_PER_POINT), key=lambda k: sub_classes[k][0])
    dms, dcnt = sub_classes[dom]
    launches_per_field = dcnt / K          # per step
    # points one launch processes: y-phase kernels and stats see the whole field; plane kernels one chunk.  With merged
    # plane launches the first substep of chan_step_filter (which shares its z-padded planes with the filter) runs the
    # separate kernels and the other two substeps the merged one.
    plane_sweeps = {"zfft_inv": 1 if merged else 3, "xfft_prod": 1 if merged else 3, "zfft_fwd": 1 if merged else 3, "planes_merged": 2}
    pts_per_launch = npts * plane_sweeps[dom] / launches_per_field if dom in plane_sweeps else npts
    abytes = BYTES_PER_POINT[dom] * pts_per_launch
    achieved = abytes / (dms / dcnt * 1e-3) / 1e9
    planes_per_launch = round(pts_per_launch / (c["nx"] * c["nz"]))
    mz_, tiles_ = 3 * c["nz"] // 2, -(-(c["nx"] // 2) // tune["tz"])
    grid = {"xfft_prod": (mz_, planes_per_launch, 1), "zfft_inv": (tiles_, planes_per_launch, 6), "zfft_fwd": (tiles_, planes_per_launch, 3)}.get(dom)
    row = ncu_row(dom, grid) if grid else None
    traffic = (float(row["dram__bytes_read.sum"]) + float(row["dram__bytes_write.sum"])) * 1e9 if row else None
    roofline = {"kernel": dom, "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic,
                "traffic_source": (f"{NCU_TABLE}, row of {row['Kernel Name'][:40]}... grid {row['Grid Size']} (ncu --set full capture of "
                                   "this round, not measured in this run)") if row else "no matching launch in " + NCU_TABLE,
                "peak_source": peak_src, "algorithmic_bytes_per_launch": abytes,
                "avg_launch_ms": dms / dcnt, "share_of_step": dms / ms_total}
    if dom == "xfft_prod":
        roofline["limiter"] = ("latency at 16 warps per SM (registers and shared memory both full with two 256-thread CTAs); "
                               "ncu: fp64 pipe 49%, issue slots 51%, L1/shared pipe 57%, DRAM 22% -- no unit saturated; the HBM "
                               "fraction is what north_star asks for, fp64 and smem are the roofs this kernel is nearer to")
        # the x pass is bound by the shared-memory pipe and the fp64 pipe, not by HBM: two more
        # roofs.  "alu": 5 N log2 N flops against the fp64 FMA rate measured by the library's register-only micro-kernel
        # (chan_debug_fma_peak) in this run; "smem": shared-memory wavefronts of one launch (ncu table) x 128 B against
        # 148 SMs x 128 B/clk x the SM clock sampled during the timed region.
        fl = xpass_flops_per_point(c["nx"], c["nz"]) * pts_per_launch
        tf = fl / (dms / dcnt * 1e-3) / 1e12
        fma_peak = ch.debug_fma_peak()
        roofline["fp64"] = {"bound": "alu", "achieved": tf, "peak": fma_peak, "unit": "TFLOP/s", "frac": tf / fma_peak, "flops_per_launch": fl,
                            "peak_source": "measured: chan_debug_fma_peak (8 independent DFMA chains per thread, 8 CTAs of 256 threads per SM)",
                            "peak_derived_note": FP64_PEAK_DERIVED_TFLOPS}
        clk_mhz = clk.summary().get("sm_mhz") or 1965.0
        if row and row.get("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum"):
            wf = float(row["l1tex__data_pipe_lsu_wavefronts_mem_shared.sum"])
            sm_peak = 148 * SMEM_BYTES_PER_CLK_PER_SM * clk_mhz * 1e6 / 1e9
            sm_ach = wf * 128 / (dms / dcnt * 1e-3) / 1e9
            roofline["smem"] = {"bound": "smem", "achieved": sm_ach, "peak": sm_peak, "unit": "GB/s", "frac": sm_ach / sm_peak,
                                "wavefronts_per_launch": wf, "peak_source": f"148 SMs x 128 B/clk x {clk_mhz:.0f} MHz (sampled)",
                                "wavefront_source": NCU_TABLE}
    groups = {}
    for gname, (classes, bpp) in SURVEY_GROUPS.items():
        if merged and gname.startswith(("K2 ", "K3 ", "K4 ")):
            continue                                         # only one of three substeps runs them separately: see the plane-phase group
        gms = sum(prof[k][0] for k in classes if k in prof)
        if gms > 0:
            gb = bpp * npts * 3 * K / (gms * 1e-3) / 1e9     # substep part only: the filter has its own classes
            groups[gname] = {"ms_per_substep": gms / (3 * K), "survey_bytes_per_point": bpp, "achieved_GBs": gb, "frac": gb / peak}
            if gname.startswith("K5+K1"):
                # the six sweeps move 384 B/point (the intermediates between dependent solves); the fraction
                # on those bytes says how close the sweeps themselves are to the roof, the one on 144 how far the design is
                moved = sum(BYTES_PER_POINT[k] for k in ("y1", "y2", "y3", "y4", "derive_down", "derive_up"))
                groups[gname]["moved_bytes_per_point"] = moved
                groups[gname]["frac_on_moved_bytes"] = moved * npts * 3 * K / (gms * 1e-3) / 1e9 / peak
    sub_gb = 432 * npts / (ms_sub / (3 * K) * 1e-3) / 1e9    # 54 field passes = 432 B/point per substep
    groups["substep total"] = {"ms_per_substep": ms_sub / (3 * K), "survey_bytes_per_point": 432, "achieved_GBs": sub_gb, "frac": sub_gb / peak}
    kernel_ms = {k: {"ms_per_step": v_[0] / K, "launches_per_step": v_[1] / K} for k, v_ in sub_classes.items()}

    # ---- end to end through the host-buffer entry points ---------------------------------------------
    e2e = None
    if rank == 0 or world > 1:
        Ke = max(1, min(args.e2e_steps, K))
        try:
            hf = torch.empty(tuple(fout.shape), dtype=torch.complex128, pin_memory=pinned)
            ch.get_state_host(hv, hp, ho, hU, hW)

            def e2e_step():
                ch.set_state_host(hv, hp, ho, hU, hW)
                ch.run(1, 1, 1, kxc, kzc, ring=fring)
                ch.stats(binding.STATS_READ)
                with torch.cuda.stream(stream):
                    hf.copy_(fout)                      # the filtered database back to pinned host memory
                ch.get_state_host(hv, hp, ho, hU, hW)

            e2e_step()
            barrier()
            t0 = time.perf_counter()
            e0.record(stream)
            for _ in range(Ke):
                e2e_step()
            e1.record(stream)
            barrier()
            wall = (time.perf_counter() - t0) * 1e3
            ms_e = max(e0.elapsed_time(e1), wall)       # host-side copies block: take the larger clock
            ms_e = max_over_ranks(ms_e, world, dev)
            state_b = 3 * F + 2 * c["ny"] * 8
            e2e = {"value": job_value(npts, 3 * Ke, world, ms_e), "unit": UNIT, "steps": Ke,
                   "ms_per_step": ms_e / Ke, "h2d_bytes_per_step": state_b,
                   "d2h_bytes_per_step": state_b + hf.numel() * 16 + 10 * c["ny"] * 8,
                   "api": "chan_set_state_host + chan_run(1 step, database + statistics) + chan_stats(READ) + database D2H + chan_get_state_host, "
                          + ("pinned" if pinned else "pageable (pinning refused)") + " host buffers"}
            del hf
        except RuntimeError as ex:      # pinned allocation refused by the host
            e2e = {"value": None, "unit": UNIT, "error": str(ex)[:200], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}

    if world > 1:
        dist.barrier()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    cufft = None
    if world == 1 and not args.no_cufft_line:
        try:
            cufft = cufft_reference_line(c, dev)
            cufft["ours_ms_per_substep"] = sum(prof[k][0] for k in ("xfft_prod", "zfft_fwd") if k in prof) / (3 * K) \
                + (prof["zfft_inv"][0] / (3 * K) if "zfft_inv" in prof else 0.0)
        except RuntimeError as ex:
            cufft = {"error": str(ex)[:200]}
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        ncores = len(os.sched_getaffinity(0))
        val, ms, sample = oracle_sample(wl, 1, 0)
        cpu = {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample, "host_cores_available": ncores}
        try:
            allv, alls = oracle_all_cores(wl, ncores)
            cpu["all_cores"] = {"value": allv, "unit": UNIT, "cores": ncores, "sample": alls}
        except Exception as ex:                    # the baseline is context: never fail the bench line over it
            cpu["all_cores"] = {"value": None, "error": str(ex)[:200]}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_total_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl, "grid": [c["nx"], c["ny"], c["nz"]], "padded": [3 * c["nx"] // 2, c["ny"], 3 * c["nz"] // 2],
                   "step": "chan_run(nsteps=1, filter_every=1, stats_every=1) = statistics + filtered database of the entry state (chan_filter_store fused into the step) + 1 RK3 step of 3 substeps; value counts the 3 substeps",
                   "filter_cut": [kxc, kzc], "l2": "inputs larger than L2 (one field = %.2f GB)" % (F / 1e9),
                   "workspace_GB": ws_bytes / 1e9, "multi_gpu": "replicas only", "state_finite": finite, "plan": plan_text,
                   "tuning": tune},
        "clocks": clk.summary(), "e2e": e2e, "gpu_launches": int(launches),
        "substep_only": substep_only, "roofline": roofline, "roofline_groups": groups, "kernel_ms": kernel_ms,
        "cpu_baseline": cpu, "cufft_reference_line": cufft,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
