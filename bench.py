#!/usr/bin/env python
"""bench.py — throughput of the overrelaxation gauge-fixing hot path (arXiv:1412.1498, Algorithm 1) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg4] [--impl ours|reference]

A STEP is one pass of the whole hot path at the workload's own cadence: `check_every` overrelaxation sweeps (each an
even and an odd half-sweep: rows a0-a5 of SURVEY.md §8(a); reunitarisation a6 where the config asks for it) followed by
one F/theta measurement (a7), i.e. one turn of the gf_fix loop (a8).  The default workload is BASELINE.json configs[4]
(64^3 x 128, FP64, 18-real links, Landau, omega = 1.8, F/theta every 20 sweeps): the largest config, the one the
roofline target is quoted on, and it fits one GPU (19.3 GB of links).  The field evolves from step to step, as it does
in the real run (W + K = 8 steps = 160 of the config's 200 sweeps).

  value      site-updates/s, links resident in HBM, CUDA events on the library's stream, max over ranks.
  e2e        the same metric through the C-ABI host entry points: every step copies the canonical field from pinned
             host memory (gf_set_links_host), runs the step, and copies the fixed field back (gf_get_links_host).
  roofline   the half-sweep kernel: algorithmic bytes per launch (16 L per site-update x V/2 sites) / mean launch
             duration measured here with CUDA events around the back-to-back half-sweep launches of each step.
  cpu_baseline / --impl reference: the CPU oracle as it stands on the box's host cores, on a bounded sample.

Multi-GPU: the path does not shard in this build ("replicas only"); --gpus N runs N independent replicas,
one process per GPU, no data-path collective; `value` is the aggregate.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "ovr_site_updates_per_s"
UNIT = "site-updates/s"
LINK_BYTES = {("f64", 18): 144, ("f64", 12): 96, ("f32", 18): 72, ("f32", 12): 48, ("f64", 8): 64, ("f32", 8): 32}
# nominal flop per site-update (add = mul = 1, FMA = 2; reconstruct + K + 3 subgroup steps + 8
# products), split into the part the kernels run in FP64 in BOTH storage precisions (K(x) and the three SU(2) steps,
# DESIGN.md §2 "Precision of the site rotation") and the part that runs in the storage precision.
# With FP64 links the rotation is FP64.  With FP32 links the staged kernels (variants 0/3/4/5/6) evaluate K(x) and the
# steps in FP32 and re-evaluate in FP64 only the sites where a subgroup's |r|^2 < 16 (FAST_TAU2 in csrc/gf_kernels.cu:
# nearly all sites of a Haar-random start, almost none once F > 0.5); the two-pass variants (1, 2) are FP64 throughout.
FLOPS_ROTATION = 144 + 597                       # K(x) + 3 subgroup steps
FLOPS_LINKS = {18: 1584, 12: 336 + 1056, 8: 1584 + 8 * 90}  # the 8 products (+ row-2 / 8-real reconstruction)
# 8-real storage: the nominal count misses what the format really costs (divisions, square roots, the decode / encode
# selects): the MEASURED FP64 warp instructions per site-update of the shipped kernel (ncu smsp__inst_executed_pipe_fp64,
# profiles/r2_8real_cfg3_ncu.txt), each counted as one FMA = 2 flop against the FMA-chain peak.
MEASURED_FP64_INSTR = {8: 2550}


def ncu_traffic(cfg_name, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on `cfg_name`, from the committed
    `ncu --set full` captures (profiles/ncu_traffic.csv names the summary each row was read from); None if absent."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(path):
        return None, None
    import csv

    best = None
    for row in csv.DictReader(l for l in open(path) if not l.startswith("#")):
        if row["config"] == cfg_name and row["kernel"] == kernel:
            best = row  # the last matching row is the newest capture
    if best is None:
        return None, None
    return float(best["dram_read_bytes"]) + float(best["dram_write_bytes"]), best["source"]


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, read+write copy)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def halfsweep_kernel_name(storage, variant, defer=False, sites_per_parity=1 << 30, prec="f64"):
    """The kernel gf_ovr_sweep launches for this storage format / GF_OPT_SWEEP_VARIANT (csrc/gf_kernels.cu, halfsweep_T)."""
    v = variant or (5 if prec == "f64" and storage != 8 and not defer else 3)
    return {1: "ovr_halfsweep_kernel", 2: "ovr_halfsweep_kernel (L2 bulk prefetch)", 3: "ovr_halfsweep_staged_kernel",
            4: "ovr_halfsweep_staged_kernel<BULK=1> (TMA bulk copies)",
            5: "ovr_halfsweep_staged_kernel<BULK=2> (forward chunk by TMA bulk copy)",
            6: "ovr_halfsweep_split_kernel (two lanes per site)"}[v] + (" (deferred temporal links)" if defer else "")


def measure_fp_peaks(seconds=0.25):
    """FP64 / FP32 FMA-chain peaks of the current device, measured now through the C ABI (gf_peak_fma)."""
    import torch

    import paper_1412_1498_b200 as gf

    scratch = torch.zeros(16, dtype=torch.uint8, device="cuda")
    out = {}
    for name, prec in (("f64_tflops", gf.GF_FP64), ("f32_tflops", gf.GF_FP32)):
        rc, t = gf.gf_peak_fma(prec, seconds, scratch.data_ptr(), torch.cuda.current_stream().cuda_stream)
        if rc != gf.GF_OK:
            raise RuntimeError(f"gf_peak_fma failed: {gf.gf_strerror(rc)}")
        out[name] = t
    out["how"] = "gf_peak_fma: register-only FMA chains (16 per thread, 8 blocks of 256 threads per SM), FMA = 2 flop"
    return out


def run_peaks(args):
    """--peaks: the measured CUDA-core peaks with the clocks seen while they ran."""
    import torch

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    measure_fp_peaks(0.05)
    sampler = ClockSampler(int(os.environ.get("LOCAL_RANK", "0")))
    fp = measure_fp_peaks(2.0)
    clocks = sampler.stop()
    hbm, src = load_peaks()
    print(json.dumps({"metric": "fma_chain_peak", "f64_tflops": fp["f64_tflops"], "f32_tflops": fp["f32_tflops"],
                      "how": fp["how"], "hbm_gbs": hbm, "hbm_source": src, "clocks": clocks,
                      "nominal": "148 SMs x 64 (FP64) / 128 (FP32) FMA lanes x 2 flop x 1.965 GHz = 37.2 / 74.5 TFLOP/s"}),
          flush=True)
    return 0


def spawn_command(gpus, argv, port=None):
    """`python bench.py --gpus N` without a launcher: the command that runs N ranks of this file, one per GPU."""
    import socket

    if port is None:
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={gpus}", "--master-addr",
            "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *argv]


def get_cfg(name):
    import gf_inputs as gi

    return dict(next(c for c in gi.CONFIGS if c["name"] == name))


def workload_name(cfg):
    d = cfg["dims"]
    return (f"BASELINE.json configs[{cfg['name'][3:]}]: {d[0]}x{d[1]}x{d[2]}x{d[3]} SU(3) {cfg['gauge']} "
            f"{cfg['prec']} {cfg['storage']}-real omega={cfg['omega']} roughness={cfg['roughness']} seed={cfg['seed']}")


# ---- clocks ------------------------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), f"--query-gpu={self.FIELDS}",
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); smax.append(float(c[2])); power.append(float(c[3]))
            except ValueError:
                continue
            for n, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            # "under load": samples in the upper half of the observed power range
            lo, hi = min(power), max(power)
            load = [s for s, p in zip(sm, power) if p >= lo + 0.5 * (hi - lo)] or sm
            load.sort()
            out.update(sm_mhz=load[len(load) // 2], sm_max_mhz=max(smax), reasons=sorted(reasons), samples=len(sm),
                       power_w_max=hi)
        return out


# ---- the oracle on host cores (cpu_baseline and --impl reference) --------------------------------------------------------
def oracle_sample_dims(cfg, slices=8):
    """A slab of the workload's lattice: same x,y,z cross-section, `slices` time slices (or the whole lattice if smaller)."""
    d = cfg["dims"]
    return (d[0], d[1], d[2], min(d[3], slices))


class OracleRun:
    """The oracle as it stands (oracle/, OpenMP over the sites of one parity) on a bounded sample of the workload."""

    def __init__(self, cfg, slices=8):
        import numpy as np

        import gf_inputs as gi
        import oracle

        self.np, self.oracle, self.cfg = np, oracle, cfg
        self.dims = oracle_sample_dims(cfg, slices)
        self.V = gi.volume(self.dims)
        dt = np.float32 if cfg["prec"] == "f32" else np.float64
        U = gi.make_links(self.dims, cfg["roughness"], cfg["seed"], dtype=dt)
        self.U = np.ascontiguousarray(U.astype(np.float64))  # reading A18: the FP64 oracle on the rounded input
        if cfg["storage"] == 12:
            oracle.project12(self.U, self.dims)
        self.cores = oracle.num_threads()
        self.sweeps_done = 0
        self.sample = (f"oracle as it stands: an unoptimised checker (g++ -O2 -ffp-contract=off, {self.cores} OpenMP "
                       f"threads), {self.dims[0]}x{self.dims[1]}x{self.dims[2]}x"
                       f"{self.dims[3]} slab of the workload lattice, same generator / gauge / storage / omega; "
                       f"one step = {cfg['check_every']} sweeps + 1 F/theta measurement (the GPU arm's cadence)")

    def step(self):
        c = self.cfg
        n = c["check_every"]
        self.oracle.sweeps(self.U, self.dims, c["gauge"], c["omega"], n=n, storage=c["storage"],
                           reunit_every=c["reunit_every"], first_sweep=self.sweeps_done)
        self.sweeps_done += n
        return self.oracle.measure(self.U, self.dims, c["gauge"])

    def time_steps(self, steps, warmup):
        for _ in range(warmup):
            self.step()
        t0 = time.perf_counter()
        for _ in range(steps):
            self.step()
        dt = time.perf_counter() - t0
        return self.V * self.cfg["check_every"] * steps / dt, dt


def run_reference(args):
    """--impl reference: the oracle timed on the host cores with the arm's metric/config.  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    if "WORLD_SIZE" in os.environ and os.environ.get("OMP_NUM_THREADS") == "1":
        # torchrun's default for its ranks; rank 0 is the only one that works here, so it takes the host's cores
        os.environ["OMP_NUM_THREADS"] = str(os.cpu_count() or 1)
    if args.oracle_threads > 0:  # before the oracle's library (and its OpenMP runtime) is loaded
        os.environ["OMP_NUM_THREADS"] = str(args.oracle_threads)
    cfg = get_cfg(args.config)
    run = OracleRun(cfg, args.oracle_slices)
    value, dt = run.time_steps(args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "sample": run.sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": run.cores, "kind": "oracle", "sample": run.sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ---- replicas: the only cross-rank traffic is the barrier and this MAX -------------------------------------
def max_over_ranks(ms_local, dist, device):
    """Elapsed time of the slowest replica.  dist = None (one process) or an initialised torch.distributed module."""
    if dist is None:
        return float(ms_local)
    import torch

    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(world, sites, sweeps, ms):
    """Whole-job site-updates/s of `world` replicas that each did `sweeps` sweeps of `sites` sites in `ms` (max)."""
    return world * sites * sweeps / (ms * 1e-3)


# ---- the CUDA path -----------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch

    import gf_inputs as gi
    import paper_1412_1498_b200 as gf

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist

        # as run_sharded: the init lines of NCCL's log let a scaling run count the ranks and see the transport chosen
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = get_cfg(args.config)
    # kernel studies on a config's lattice (secondary lines, named in config.workload): another storage format, Coulomb
    # gauge, deferred temporal links
    if args.storage:
        cfg["storage"] = args.storage
    if args.gauge:
        cfg["gauge"] = args.gauge
    if args.prec:
        cfg["prec"] = args.prec
    dims, prec, storage = cfg["dims"], cfg["prec"], cfg["storage"]
    V = gi.volume(dims)
    L = LINK_BYTES[(prec, storage)]
    n_sw = cfg["check_every"]
    omega = cfg["omega"]

    N = args.ncolors or 3
    if N != 3:  # general SU(N) study (gf_create_sun): all N^2 entries stored, host generator, no e2e / CPU legs
        import numpy as np

        args.no_e2e = args.no_cpu = True
        storage = 2 * N * N
        L = storage * (8 if prec == "f64" else 4)
        fx = gf.GaugeFixer(dims, gauge=cfg["gauge"], prec=prec, ncolors=N, device=f"cuda:{local}")
    else:
        fx = gf.GaugeFixer(dims, gauge=cfg["gauge"], prec=prec, storage=storage, device=f"cuda:{local}")
    if args.defer:
        fx.defer_temporal_links()
    if storage == 8 and N == 3:  # a study on a rough synthetic field: a few of its 1.3e8 links lie outside the format's domain
        fx.set_option(gf.GF_OPT_DOMAIN8_CHECK, 0)
    if args.variant:
        fx.set_option(gf.GF_OPT_SWEEP_VARIANT, args.variant)
    if args.block:
        fx.set_option(gf.GF_OPT_BLOCK_THREADS, args.block)
    fx.set_reunit_every(cfg["reunit_every"])
    if N != 3:
        canon = torch.from_numpy(gi.make_links_sun(dims, N, cfg["roughness"], cfg["seed"] + 1000 * rank,
                                                   dtype=np.float64 if prec == "f64" else np.float32)).cuda()
    else:
        canon = fx.new_links_buffer()
        gi.make_links_device(canon.data_ptr(), dims, cfg["roughness"], cfg["seed"] + 1000 * rank, prec,
                             torch.cuda.current_stream().cuda_stream)
    fx.set_links(canon)
    torch.cuda.synchronize()

    ev = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731  (the library runs on torch's current stream)

    def step(timers=None):
        if timers is None:
            fx.ovr_sweep(n_sw, omega)
            return fx.measure()
        a, b, c = ev(), ev(), ev()
        a.record()
        fx.ovr_sweep(n_sw, omega)
        b.record()
        r = fx.measure()  # synchronises the stream
        c.record()
        timers.append((a, b, c))
        return r

    # ---- device-resident timing (SURVEY.md 8(d) "Timing protocol"): --reps repetitions, each from a fresh gf_set_links:
    # W warm-up steps, then exactly K steps between barriers.  The line reports the MEDIAN repetition (all of its
    # numbers: value, ms_per_step, roofline, clocks, launch count) with the minimum and every repetition beside it.
    def timed_repetition():
        fx.set_links(canon)
        torch.cuda.synchronize()
        for _ in range(args.warmup):
            step()
        barrier()
        sampler = ClockSampler(local)
        launches0 = fx.kernel_launches()
        timers = []
        t0, t1 = ev(), ev()
        t0.record()
        for _ in range(args.steps):
            F, th = step(timers)
        t1.record()
        barrier()
        rep = {"launches": fx.kernel_launches() - launches0, "clocks": sampler.stop(), "F": F, "th": th,
               "ms_sweeps": sum(a.elapsed_time(b) for a, b, _ in timers),
               "ms_measure": sum(b.elapsed_time(c) for _, b, c in timers)}
        rep["ms_total"] = max_over_ranks(t0.elapsed_time(t1), dist, "cuda")
        return rep

    reps = [timed_repetition() for _ in range(max(1, args.reps))]
    by_time = sorted(reps, key=lambda r: r["ms_total"])
    med = by_time[(len(by_time) - 1) // 2]  # the median (lower of the middle two for an even count)
    launches, clocks, F, th = med["launches"], med["clocks"], med["F"], med["th"]
    ms_total, ms_sweeps, ms_measure = med["ms_total"], med["ms_sweeps"], med["ms_measure"]
    n_reunit = 0 if not cfg["reunit_every"] else sum(
        1 for s in range((args.warmup) * n_sw + 1, (args.warmup + args.steps) * n_sw + 1) if s % cfg["reunit_every"] == 0)
    value = aggregate_value(world, V, n_sw * args.steps, ms_total)
    repetitions = {"n": len(reps), "what": "each repetition: fresh gf_set_links, %d warm-up steps, %d timed steps; value / "
                   "ms_per_step / roofline are the median repetition's" % (args.warmup, args.steps),
                   "values": [aggregate_value(world, V, n_sw * args.steps, r["ms_total"]) for r in reps],
                   "median": value, "max": aggregate_value(world, V, n_sw * args.steps, by_time[0]["ms_total"]),
                   "min": aggregate_value(world, V, n_sw * args.steps, by_time[-1]["ms_total"]),
                   "ms_per_step": [r["ms_total"] / args.steps for r in reps]}

    # ---- roofline of the dominant kernel (half-sweep): 2*n_sw launches per step, back to back on the stream
    peak, peak_src = load_peaks()
    n_half = 2 * n_sw * args.steps
    bytes_per_launch = (14 if args.defer else 16) * L * (V // 2)  # deferred: 6 links + the accumulator, read and written
    # the reunitarisation launches inside the sweep region (config 2 only) are subtracted at their algorithmic cost
    ms_half = (ms_sweeps - n_reunit * (8 * V * L) / (peak * 1e9) * 1e3) / n_half
    achieved = bytes_per_launch / (ms_half * 1e-3) / 1e9
    kernel = halfsweep_kernel_name(storage, args.variant, args.defer, V // 2, prec) if N == 3 else f"halfsweep_sun_kernel<N={N}>"
    traffic, traffic_src = ncu_traffic(cfg["name"], kernel) if not (args.storage or args.gauge or args.defer or args.prec or N != 3) else (None, None)
    # flops leg: the FMA-chain peaks measured now, on this GPU, under the clocks it runs at after
    # the timed region (gf_peak_fma); the site rotation is FP64 in both storage precisions, the link products are in
    # the storage precision
    fp = measure_fp_peaks(0.25)
    flops_source, flops64_slow_path = "SURVEY.md 8(d), nominal counts", None
    if N == 3 and prec == "f64" and storage in MEASURED_FP64_INSTR:
        flops64, flops32 = 2 * MEASURED_FP64_INSTR[storage], 0
        flops_source = "measured FP64 warp instructions per site-update x 2 (profiles/r2_8real_cfg3_ncu.txt)"
    elif N == 3:
        fast32 = prec == "f32" and args.variant in (0, 3, 4, 5, 6)  # site rotation on the FP32 units (fast path)
        flops64 = (0 if fast32 else FLOPS_ROTATION) + (FLOPS_LINKS[storage] if prec == "f64" else 0)
        flops32 = (FLOPS_ROTATION if fast32 else 0) + (FLOPS_LINKS[storage] if prec == "f32" else 0)
        if fast32:  # a site below FAST_TAU2 pays the FP32 attempt and the FP64 re-evaluation
            flops64_slow_path = FLOPS_ROTATION
            flops_source += "; rotation counted on the FP32 fast path (flops_leg_ms_all_sites_reevaluated: every site " \
                            "also takes the FP64 branch, the Haar-random start)"
    else:  # the same counting for N x N: K sum, N(N-1)/2 subgroup steps (31 + two 2-row rotations), 8 full products
        rot = 8 * 2 * N * N + (N * (N - 1) // 2) * (31 + 2 * 14 * N)
        prod = 8 * N * N * (8 * N - 2)
        flops64, flops32 = rot + (prod if prec == "f64" else 0), (prod if prec == "f32" else 0)
    t_bytes_ms = bytes_per_launch / (peak * 1e9) * 1e3
    t_flops_ms = (V // 2) * (flops64 / (fp["f64_tflops"] * 1e12) + flops32 / (fp["f32_tflops"] * 1e12)) * 1e3
    roofline = {"bound": "hbm" if t_bytes_ms >= t_flops_ms else "alu", "kernel": kernel, "achieved": achieved, "peak": peak,
                "unit": "GB/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": peak_src,
                "peak_note": "a read+write copy, the same 50/50 mix as this kernel; frac > 1 means the kernel moves its "
                             "bytes faster than torch's copy does, not that it beats the memory system (read-only passes "
                             "reach 7.3-7.4 TB/s on this part, HBM3e nominal is 7.7-8 TB/s)",
                "algorithmic_bytes_per_launch": bytes_per_launch, "ms_per_launch": ms_half,
                "roofline_ms_per_launch": max(t_bytes_ms, t_flops_ms), "bytes_leg_ms": t_bytes_ms, "flops_leg_ms": t_flops_ms,
                "frac_of_roofline_time": max(t_bytes_ms, t_flops_ms) / ms_half,
                "flops_per_site_update": {"fp64": flops64, "fp32": flops32, "source": flops_source},
                "fp_peaks": fp,
                "launches_timed": n_half, "share_of_step": ms_sweeps / ms_total,
                "measure_ms": ms_measure / args.steps,
                "measure_gbs": 4 * V * L / (ms_measure / args.steps * 1e-3) / 1e9,
                "whole_step_gbs": (16 * V * L * n_sw + 4 * V * L) / (ms_total / args.steps * 1e-3) / 1e9}
    roofline["whole_step_frac"] = roofline["whole_step_gbs"] / peak
    if flops64_slow_path is not None:
        roofline["flops_leg_ms_all_sites_reevaluated"] = t_flops_ms + (V // 2) * flops64_slow_path / (fp["f64_tflops"] * 1e12) * 1e3

    # ---- the config's whole contract run (gf_fix from fresh links with the config's eps / sweep cap / cadence):
    # config 4's "fixed 200 sweeps with F/theta every 20 sweeps, run as a sustained-throughput test"
    contract = None
    if not args.no_contract:
        fx.set_links(canon)
        torch.cuda.synchronize()
        c0, c1 = ev(), ev()
        c0.record()
        done = fx.fix(omega, cfg["eps"], cfg["max_sweeps"], n_sw)
        c1.record()
        torch.cuda.synchronize()
        ms_c = max_over_ranks(c0.elapsed_time(c1), dist, "cuda")
        hist = fx.history()
        contract = {"what": f"gf_fix(omega={omega}, eps={cfg['eps']}, max_sweeps={cfg['max_sweeps']}, check_every={n_sw})",
                    "sweeps_done": done, "measurements": len(hist), "ms": ms_c,
                    "value": aggregate_value(world, V, done, ms_c), "unit": UNIT,
                    "final_F": hist[-1][1], "final_theta": hist[-1][2]}

    # ---- end to end through the host entry points (pinned host memory, copies inside the timed region)
    e2e = None
    nbytes = V * 72 * (8 if prec == "f64" else 4)

    def host_mem_available():
        try:
            return int(next(l for l in open("/proc/meminfo") if l.startswith("MemAvailable")).split()[1]) * 1024
        except (OSError, StopIteration):
            return 0

    # every rank of the node pins its own copy of the field: leave the leg out (on all ranks alike) rather than run the
    # host out of memory
    e2e_fits = host_mem_available() > 1.25 * world * nbytes
    if dist is not None:
        flag = torch.tensor([1.0 if e2e_fits else 0.0], device="cuda")
        dist.all_reduce(flag, op=dist.ReduceOp.MIN)
        e2e_fits = bool(flag.item() > 0.5)
    if not args.no_e2e and not e2e_fits:
        log(f"bench.py: e2e leg left out: {world} x {nbytes / 1e9:.1f} GB of pinned host memory do not fit")
        e2e = {"value": None, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes + 16,
               "skipped": "not enough host memory to pin one field per rank"}
    if not args.no_e2e and e2e_fits:
        host = torch.empty((V, 4, 3, 3, 2), dtype=fx.dtype).pin_memory()
        host.copy_(canon)
        del canon
        torch.cuda.empty_cache()
        n_e2e = max(1, min(args.steps, args.e2e_steps))

        # Two fields in flight (a user fixing a stream of configurations): a second context on its own stream with its
        # own pinned buffer, driven by a second host thread, so that one field's upload overlaps the other's sweeps or
        # download (PCIe is full duplex, the GPU has separate copy engines).  Every step of every lane still uploads
        # its inputs and downloads its result inside the timed region.
        lanes = [(fx, host)]
        avail = host_mem_available() / world  # this rank's share of what is left
        while len(lanes) < args.e2e_lanes and avail > 2 * nbytes and \
                torch.cuda.mem_get_info()[0] > 1.3 * nbytes:
            try:  # a lane that cannot get its memory is left out; the leg then runs with the lanes it has
                s2 = torch.cuda.Stream()
                fx2 = gf.GaugeFixer(dims, gauge=cfg["gauge"], prec=prec, storage=storage, device=f"cuda:{local}", stream=s2)
                fx2.set_reunit_every(cfg["reunit_every"])
                host2 = torch.empty((V, 4, 3, 3, 2), dtype=fx.dtype).pin_memory()
                host2.copy_(host)
            except (RuntimeError, MemoryError) as err:
                log(f"bench.py: e2e lane {len(lanes) + 1} not created ({err})")
                break
            lanes.append((fx2, host2))

        import threading

        # one upload and one download at a time: two copies in the same direction would only share the bus
        up_lock, down_lock = threading.Lock(), threading.Lock()

        def e2e_step(lane, uploaded=None):
            f, h = lane
            with up_lock:
                f.set_links_host(h)
            if uploaded is not None:
                uploaded.set()
            f.ovr_sweep(n_sw, omega)
            r = f.measure()
            with down_lock:
                f.get_links_host(h)
            return r

        def run_lanes(n):
            # lane k starts once lane k-1 has finished its first upload: the lanes run out of phase, so one lane's
            # upload meets another's download instead of its upload
            gates = [threading.Event() for _ in lanes]

            def work(k):
                torch.cuda.set_device(local)
                if k > 0:
                    gates[k - 1].wait()
                for i in range(n):
                    e2e_step(lanes[k], gates[k] if i == 0 else None)

            ts = [threading.Thread(target=work, args=(k,)) for k in range(1, len(lanes))]
            for t in ts:
                t.start()
            work(0)
            for t in ts:
                t.join()

        run_lanes(1)  # warm-up
        barrier()
        w0 = time.perf_counter()
        run_lanes(n_e2e)
        barrier()
        ms_e2e = (time.perf_counter() - w0) * 1e3  # wall clock around synchronising calls on several streams
        ms_e2e = max_over_ranks(ms_e2e, dist, "cuda")
        steps_done = n_e2e * len(lanes)
        e2e = {"value": aggregate_value(world, V, n_sw * steps_done, ms_e2e), "unit": UNIT, "h2d_bytes_per_step": nbytes,
               "d2h_bytes_per_step": nbytes + 16, "steps": steps_done, "ms_per_step": ms_e2e / steps_done,
               "lanes": len(lanes),
               "what": "%s: each step is gf_set_links_host (pinned) + %d sweeps + gf_measure + gf_get_links_host "
                       "(pinned) of one field on its own context, stream and host thread"
                       % ("throughput of a stream of configurations with %d fields in flight (not the latency of one)"
                          % len(lanes) if len(lanes) > 1 else "one field at a time", n_sw)}
        for f, h in lanes[1:]:
            f.close()
        lanes = None
        del host
    fx.close()

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- the oracle beside it, on this box's host cores (rank 0, N = 1 only)
    cpu = None
    if world == 1 and not args.no_cpu:
        run = OracleRun(cfg)
        v, dt = run.time_steps(1, 0)
        cpu = {"value": v, "unit": UNIT, "cores": run.cores, "kind": "oracle", "sample": run.sample, "seconds": dt}
        # SURVEY.md 8(d) "Oracle timed beside it": once with all cores (above) and once with ONE thread, in a process of
        # its own (the OpenMP runtime takes its thread count when the oracle's library is loaded), on a two-slice slab so
        # that the leg stays near ten seconds
        try:
            r = subprocess.run([sys.executable, os.path.abspath(__file__), "--impl", "reference", "--config", cfg["name"],
                                "--steps", "1", "--warmup", "0", "--oracle-threads", "1", "--oracle-slices", "2"],
                               capture_output=True, text=True, timeout=600,
                               env={k: v_ for k, v_ in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")})
            one = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][-1])
            cpu["one_thread"] = {"value": one["value"], "unit": UNIT, "cores": one["cpu_baseline"]["cores"],
                                 "sample": one["cpu_baseline"]["sample"], "seconds": one["ms_per_step"] * 1e-3}
        except Exception as exc:  # a reported baseline, never a reason to lose the GPU line
            cpu["one_thread"] = {"unavailable": repr(exc)[:200]}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": prec, "data": "synthetic",
        "config": {"workload": workload_name(cfg) + (" (deferred temporal links)" if args.defer else "") + (f" [study: SU({N}) links, all N^2 entries stored]" if N != 3 else "")
                   + (" [study: not the config's own storage / gauge / precision]" if args.storage or args.gauge or args.prec else ""),
                   "step": f"{n_sw} sweeps + 1 F/theta measurement",
                   "sites": V, "l2": "inputs exceed L2 (field %.2f GB vs 126 MB)" % (4 * V * L / 1e9)
                   if 4 * V * L > 4 * 126e6 else "field fits L2: not an HBM measurement", "parallelism": "replicas only",
                   "final_F": F, "final_theta": th},
        "roofline": roofline, "contract_run": contract, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "repetitions": repetitions,
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def run_fftsd(args):
    """--algo fftsd: Algorithm 2 (steepest descent with Fourier acceleration) on the same workload.
    A step = `check_every` iterations (Delta+F/theta pass, transforms + factor + inverse transforms, rotation) + one read
    of F/theta.  Secondary line: metric fftsd_site_iterations_per_s, not the headline."""
    import torch

    import gf_inputs as gi
    import paper_1412_1498_b200 as gf

    cfg = get_cfg(args.config)
    dims, prec, storage = cfg["dims"], cfg["prec"], cfg["storage"]
    V = gi.volume(dims)
    L = LINK_BYTES[(prec, storage)]
    n_it = cfg["check_every"]
    fx = gf.GaugeFixer(dims, gauge=cfg["gauge"], prec=prec, storage=storage)
    canon = fx.new_links_buffer()
    gi.make_links_device(canon.data_ptr(), dims, cfg["roughness"], cfg["seed"], prec,
                         torch.cuda.current_stream().cuda_stream)
    fx.set_links(canon)
    del canon
    fx.fft_attach()
    torch.cuda.synchronize()
    for _ in range(args.warmup):
        fx.fft_step(n_it, 0.08)
        fx.measure()
    torch.cuda.synchronize()
    l0 = fx.kernel_launches()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    for _ in range(args.steps):
        fx.fft_step(n_it, 0.08)
        F, th = fx.measure()
    t1.record()
    torch.cuda.synchronize()
    ms = t0.elapsed_time(t1)
    peak, peak_src = load_peaks()
    csize = 16 if prec == "f64" else 8
    # algorithmic bytes per iteration: Delta pass reads 4VL, writes 4 fields; rotation reads+writes 4VL and reads the
    # fields; each transform pass and the factor read+write the 4 fields (3-D: 1 pass, +1 for t in Landau gauge)
    passes = 2 * (2 if cfg["gauge"] == "landau" else 1) + 1
    bytes_it = 12 * V * L + 4 * V * csize * (2 + 2 * passes)
    gbs = bytes_it * n_it * args.steps / (ms * 1e-3) / 1e9
    line = {"metric": "fftsd_site_iterations_per_s", "value": V * n_it * args.steps / (ms * 1e-3),
            "unit": "site-iterations/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": prec, "data": "synthetic",
            "config": {"workload": workload_name(cfg), "algorithm": "Algorithm 2, alpha=0.08",
                       "step": f"{n_it} iterations + 1 F/theta measurement", "final_F": F, "final_theta": th},
            "roofline": {"bound": "hbm", "kernel": "whole iteration (sd_delta, transform passes with the Fourier factor, sd_rotate)",
                         "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
                         "traffic": ncu_traffic(cfg["name"], "fftsd_iteration")[0],
                         "peak_source": peak_src, "algorithmic_bytes_per_iteration": bytes_it},
            "gpu_launches": int(fx.kernel_launches() - l0)}
    fx.close()
    if not args.no_cpu:  # the numpy oracle of Algorithm 2 as it stands, on a slab of the same lattice
        import numpy as np

        from oracle import fftsd

        sd = oracle_sample_dims(cfg)
        Uo = np.ascontiguousarray(gi.make_links(sd, cfg["roughness"], cfg["seed"]))
        w0 = time.perf_counter()
        fftsd.step(Uo, sd, cfg["gauge"], 0.08, storage=storage)
        F, th = fftsd.measure(Uo, sd, cfg["gauge"])
        dt = time.perf_counter() - w0
        line["cpu_baseline"] = {"value": gi.volume(sd) / dt, "unit": "site-iterations/s", "cores": os.cpu_count(),
                                "kind": "oracle", "seconds": dt,
                                "sample": f"oracle/fftsd.py (numpy, FP64), 1 iteration + 1 F/theta on a "
                                          f"{sd[0]}x{sd[1]}x{sd[2]}x{sd[3]} slab of the workload lattice"}
    print(json.dumps(line), flush=True)
    return 0


HALO_HOW = {"flags": "stored by the border kernel into the neighbour's workspace (same process: plain pointer, other rank: "
                     "CUDA-IPC mapping); neighbours ordered by stream-ordered flag writes / waits; the sweep is one libgf call",
            "ipc": "stored by the border kernel into the CUDA-IPC mapped workspace of the neighbour rank; one 1-element "
                   "all-reduce per half-sweep orders the ranks",
            "events": "stored by the border kernel into the neighbour slab of the same process; kernels ordered by CUDA events",
            "transport": "NCCL send/recv between ranks, device copies within a rank"}


def run_sharded(args):
    """--sharded K: the overrelaxation sweep over T-slabs (paper_1412_1498_b200.sharded; SURVEY.md §8(f) NEXT-2,
    PAPER.md:132-134).  The paper's weak-scaling point (32^4 per GPU) is
        python bench.py --gpus N --sharded 1 --config cfg2
    (unmeasured on more than one GPU: this pool leases one).  Every rank holds the config's lattice as K slabs; the global lattice is world x taller (fixed
    local volume per GPU, the paper's weak-scaling set-up).  Secondary line: with one rank the halo
    messages are device-to-device copies and the number is the cost of the border / interior split on one GPU."""
    import torch

    import gf_inputs as gi
    import paper_1412_1498_b200 as gf

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist

        # NCCL's initialisation lines stay on (stderr), so that a reader of the log can count the ranks and see the transport
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg = get_cfg(args.config)
    dims, prec, storage = cfg["dims"], cfg["prec"], cfg["storage"]
    K = args.sharded
    gdims = (dims[0], dims[1], dims[2], dims[3] * world)
    n_slabs = K * world
    V = gi.volume(dims)
    L = LINK_BYTES[(prec, storage)]
    n_sw, omega = cfg["check_every"], cfg["omega"]
    sh = gf.ShardedGaugeFixer(gdims, n_slabs, gauge=cfg["gauge"], prec=prec, storage=storage, device=f"cuda:{local}",
                              mode=args.sharded_mode or ("transport" if args.no_direct else None))
    sh.set_reunit_every(cfg["reunit_every"])
    if args.force_flags:  # what a rank of a multi-rank run executes, timed in one process
        for e in sh.engines.values():
            e.fx.set_option(gf.GF_OPT_SLAB_FORCE_FLAGS, 1)
    links = {}
    for s in sh.slabs:  # every slab its own seeded field of the config's recipe (rougher across slab boundaries)
        e = sh.engines[s]
        buf = e.fx.new_links_buffer()
        gi.make_links_device(buf.data_ptr(), sh.local_dims, cfg["roughness"], cfg["seed"] + 1000 * s, prec,
                             torch.cuda.current_stream().cuda_stream)
        links[s] = buf
    sh.set_links(links)
    del links, buf
    torch.cuda.synchronize()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        sh.ovr_sweep(n_sw, omega)
        sh.measure()
    barrier()
    l0 = sh.kernel_launches()
    sampler = ClockSampler(local) if rank == 0 else None
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    for _ in range(args.steps):
        sh.ovr_sweep(n_sw, omega)
        F, th = sh.measure()
    t1.record()
    barrier()
    ms = max_over_ranks(t0.elapsed_time(t1), dist, f"cuda:{local}")
    clocks = sampler.stop() if sampler else None
    if rank == 0:
        peak, peak_src = load_peaks()
        value = aggregate_value(world, V, n_sw * args.steps, ms)
        gbs = value / world * 16 * L / 1e9  # per GPU and site-update: 8 links read and written
        halo = sum(e.halo_bytes for e in sh.engines.values())
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": prec, "data": "synthetic",
                "config": {"workload": workload_name(cfg) + f" per GPU; global lattice {gdims[0]}x{gdims[1]}x{gdims[2]}x{gdims[3]}",
                           "step": f"{n_sw} sweeps + 1 F/theta measurement",
                           "parallelism": f"T-slabs: {n_slabs} slabs over {world} rank(s), {K} per rank",
                           "halo": f"2 messages of {halo // len(sh.engines)} B per slab and half-sweep "
                                   f"({HALO_HOW[sh.mode] if world > 1 or sh.mode != 'transport' else 'device copies'})",
                           "mode": sh.mode,
                           "l2": "inputs exceed L2" if 4 * V * L > 126e6 else "field fits L2 in part",
                           "final_F": F, "final_theta": th},
                "roofline": {"bound": "hbm", "kernel": "ovr_halfsweep_staged_kernel (border + interior launches)",
                             "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "traffic": None,
                             "peak_source": peak_src, "note": "whole step incl. halo traffic and measurement"},
                "gpu_launches": int(sh.kernel_launches() - l0), "halo_copies": sh.copies,
                "halo_messages_sent": sh.messages_sent, "clocks": clocks}
        print(json.dumps(line), flush=True)
    sh.close()
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--reps", type=int, default=3,
                    help="repetitions of the timed region, each from a fresh gf_set_links (the line reports the median)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg4", help="cfg0..cfg4 of BASELINE.json (default: the largest, cfg4)")
    ap.add_argument("--variant", type=int, default=0, help="GF_OPT_SWEEP_VARIANT (kernel studies)")
    ap.add_argument("--block", type=int, default=0, help="GF_OPT_BLOCK_THREADS (kernel studies)")
    ap.add_argument("--e2e-steps", type=int, default=4, help="end-to-end steps per lane")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-lanes", type=int, default=2,
                    help="fields in flight in the end-to-end leg (measured on cfg4: 1 lane 0.69 G, 2 lanes 1.00 G, 4 lanes 1.05 G)")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-contract", action="store_true", help="skip the timed whole-config gf_fix run")
    ap.add_argument("--algo", default="ovr", choices=["ovr", "fftsd"], help="ovr = Algorithm 1 (headline); fftsd = Algorithm 2")
    ap.add_argument("--sharded", type=int, default=0, metavar="K",
                    help="T-slab sharded sweep with K slabs per rank (secondary line; default 0 = single context / replicas)")
    ap.add_argument("--storage", type=int, default=0, help="kernel study: 18, 12 or 8 (FP64) instead of the config's storage")
    ap.add_argument("--gauge", default="", choices=["", "landau", "coulomb"], help="kernel study: another gauge on the config's lattice")
    ap.add_argument("--prec", default="", choices=["", "f64", "f32"], help="kernel study: another precision on the config's lattice")
    ap.add_argument("--ncolors", type=int, default=0, choices=[0, 2, 3, 4],
                    help="kernel study: SU(N) links (gf_create_sun) on the config's lattice, host generator (use cfg2 or smaller)")
    ap.add_argument("--defer", action="store_true", help="kernel study: Coulomb gauge with deferred temporal links (gf_defer_*)")
    ap.add_argument("--no-direct", action="store_true", help="--sharded: halo messages through the transport even in one process")
    ap.add_argument("--force-flags", action="store_true",
                    help="--sharded: signal / wait through the flags even where one stream orders all slabs")
    ap.add_argument("--sharded-mode", default="", choices=["", "flags", "ipc", "events", "transport"],
                    help="--sharded: ShardedGaugeFixer mode (default: flags on GPUs)")
    ap.add_argument("--oracle-threads", type=int, default=0, help="--impl reference: OpenMP threads of the oracle (0 = all cores)")
    ap.add_argument("--oracle-slices", type=int, default=8, help="--impl reference: time slices of the oracle's sample slab")
    ap.add_argument("--peaks", action="store_true", help="print the measured FP64 / FP32 FMA-chain peaks and exit")
    args = ap.parse_args()
    if args.peaks:
        return run_peaks(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started without a launcher: become N ranks, one per GPU (the driver's torchrun line does the same)
        return subprocess.call(spawn_command(args.gpus, sys.argv[1:]))
    if args.impl == "reference":
        return run_reference(args)
    if args.sharded:
        return run_sharded(args)
    if args.algo == "fftsd":
        return run_fftsd(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
