#!/usr/bin/env python
"""bench.py — throughput of the gauge-fixing hot path on B200 (contract: see DESIGN.md §9).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

Workload (BASELINE.json configs[4], the configuration the metric is quoted on): Landau gauge
overrelaxation omega = 1.7 on a 64^3 x 256 lattice, DP / 18 reals (headline line) and, as
`variants`, SP-18, SP-12, DP-12 and MP-12 on the same lattice.  One *step* = one gf_run call of
SWEEPS_PER_STEP (100) sweeps = 200 half-sweep kernels, the DP reunitarisation that falls due every
100 sweeps in the SP/MP modes, and one F/theta device reduction (the whole hot path,
SURVEY.md §8(a)).  Inputs are synthetic: the eps = 0.5 random-algebra lattice with a
Haar gauge transform of configs[1]'s recipe on a 16^4 tile, tiled periodically to the full extent
(the sweep's cost is data independent).

`value` is timed with CUDA events on the context's stream with the links resident in HBM; `e2e`
repeats the same steps through the C ABI with pinned HOST buffers: gf_set_links (host -> device) +
gf_run + gf_get_links (device -> host) inside the timed region.  `roofline` is the half-sweep
kernel: algorithmic bytes (every touched link read once and written once, 2*8*R*s bytes per site
update) divided by its mean launch duration measured with CUDA events inside the timed region.
`cpu_baseline` is the oracle (oracle/gf_oracle.cpp, as it stands) on the host cores on a bounded
sample; `--impl reference` times that oracle alone.  N > 1 runs N independent replicas, one lattice
per GPU ("replicas only"): there is no data-path collective.
"""
from __future__ import annotations

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

import numpy as np

LANDAU, OR = 0, 0
OMEGA = 1.7
SWEEPS_PER_STEP = 100
TILE = (16, 16, 16, 16)            # (Nx, Ny, Nz, Nt) of the generated tile
TILE_EPS, TILE_SEEDS = 0.5, (1004, 2004)
PREC_NAMES = {"sp": 0, "dp": 1, "mp": 2}
DTYPE_NAMES = {"sp": "f32", "dp": "f64", "mp": "f32 (Step 1 in f64)"}

# dram__bytes_read.sum + dram__bytes_write.sum per half-sweep launch from the `ncu --set full`
# captures summarised under profiles/ (bytes; key = (workload, precision, recon, "NxxNyxNzxNt"), workload = "or" for
# the overrelaxation kernels).  The file names the commit whose kernels were captured: it has to be regenerated when a
# kernel changes, and the bench line says which capture it quotes.
NCU_TRAFFIC, NCU_TRAFFIC_COMMIT = {}, None
try:
    with open(os.path.join(ROOT, "profiles", "traffic.csv")) as _fh:
        for _line in _fh:
            if _line.startswith("# captured_at_commit:"):
                NCU_TRAFFIC_COMMIT = _line.split(":", 1)[1].strip()
            _f = _line.strip().split(",")
            if len(_f) >= 4 and not _line.startswith("#"):
                _wl = _f[8] if len(_f) > 8 else "or"
                _prec = _f[0].split("_")[-1]
                if _prec in PREC_NAMES:
                    NCU_TRAFFIC[("or" if _wl.startswith("or") else _wl, _prec, int(_f[1]), _f[2])] = float(_f[3])
except OSError:
    pass


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--lattice", default="64,64,64,256", help="Nx,Ny,Nz,Nt")
    ap.add_argument("--precision", default="dp", choices=list(PREC_NAMES))
    ap.add_argument("--recon", type=int, default=18, choices=[12, 18])
    ap.add_argument("--gauge", default="landau", choices=["landau", "coulomb", "mag"], help="side study: gauge of the headline line")
    ap.add_argument("--algo", default="or", choices=["or", "sr", "sa", "micro"], help="side study: update rule of the headline line")
    ap.add_argument("--param", type=float, default=OMEGA, help="omega | p | T of --algo")
    ap.add_argument("--group", default="su3", choices=["su3", "su2"],
                    help="gauge group of the headline line (su2: side study, GF_FLAG_SU2, 4 reals per link)")
    ap.add_argument("--sweeps-per-step", type=int, default=SWEEPS_PER_STEP)
    ap.add_argument("--no-variants", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-others", action="store_true", help="skip the 32^3x64 and batched-copies side measurements")
    ap.add_argument("--block", type=int, default=0, help="CTA size override of the half-sweep kernel (tuning)")
    ap.add_argument("--shard-t", action="store_true",
                    help="N > 1: ONE lattice split along t over the N GPUs (t-shards, DESIGN.md §10; strong scaling) "
                         "instead of N independent replicas")
    return ap.parse_args()


def peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def bytes_per_site_update(prec: str, recon: int, nd: int = 4) -> int:
    """Algorithmic HBM bytes per site update: 2*nd links read once + written once."""
    s = 8 if prec == "dp" else 4
    return 2 * (2 * nd) * recon * s


# ---- clocks ---------------------------------------------------------------------------------
class ClockSampler:
    QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
             "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line)

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); smax.append(float(f[2])); power.append(float(f[3]))
            except ValueError:
                continue
            for name, v in zip(self.NAMES, f[5:9]):
                if v == "Active":
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(smax), "power_w_max": max(power),
                "samples": len(sm), "reasons": sorted(reasons)}


# ---- inputs ---------------------------------------------------------------------------------
def make_tile():
    from paper_1212_5221_b200 import inputs
    U = inputs.make_config(*TILE, TILE_EPS, *TILE_SEEDS)      # complex [Nt,Nx,Ny,Nz,4,3,3]
    return inputs.as_real(U, np.float64)


def reps_for(dims_xyzt):
    Nx, Ny, Nz, Nt = dims_xyzt
    tx, ty, tz, tt = TILE
    for n, t in ((Nx, tx), (Ny, ty), (Nz, tz), (Nt, tt)):
        if n % t:
            raise SystemExit(f"lattice extent {n} is not a multiple of the {t}-site tile")
    return (Nt // tt, Nx // tx, Ny // ty, Nz // tz)


# ---- the oracle legs (cpu_baseline, --impl reference) ------------------------------------------
ORACLE_SAMPLE_DIMS = (32, 32, 32, 64)    # Nx,Ny,Nz,Nt: a 1/32 sample of the 64^3 x 256 workload


def oracle_leg(tile, prec: str, sweeps_per_step: int, steps: int, warmup: int):
    """Times the oracle as it stands on a bounded sample of the same workload."""
    from oracle import gf_oracle as O
    from paper_1212_5221_b200 import inputs
    r = reps_for(ORACLE_SAMPLE_DIMS)
    dt = np.float64 if prec == "dp" else np.float32
    L = np.ascontiguousarray(inputs.tile_lattice(tile, r + (1,)).astype(dt))
    V = L.size // 72

    def step():
        for s in range(sweeps_per_step):
            O.sweep(L, O.LANDAU, O.OR, OMEGA, 0, s, prec == "mp")
        if prec != "dp":
            O.reunitarize(L)
        return O.measure(L, O.LANDAU)

    for _ in range(warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(steps):
        m = step()
    dt_s = time.perf_counter() - t0
    return {"value": V * sweeps_per_step * steps / dt_s, "seconds": dt_s, "cores": O.num_threads(), "V": V,
            "F": m["F"], "theta": m["theta"]}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    dims = tuple(int(x) for x in args.lattice.split(","))
    sps = 5                                   # sweeps per reference step: bounded sample
    tile = make_tile()
    r = oracle_leg(tile, args.precision, sps, args.steps, args.warmup)
    sample = (f"{args.steps} steps x {sps} Landau OR sweeps (+1 F/theta measurement) of the CPU oracle on a "
              f"{'x'.join(map(str, ORACLE_SAMPLE_DIMS))} sample (V={r['V']}) of the {args.lattice} workload")
    line = {
        "impl": "reference", "metric": "site-updates/s (Landau OR sweep incl. F/theta reductions)",
        "value": r["value"], "unit": "site-updates/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * r["seconds"] / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": DTYPE_NAMES[args.precision], "data": "synthetic",
        "config": {"workload": f"Landau OR omega=1.7, {'x'.join(map(str, dims))} (BASELINE.json configs[4]), "
                               f"{args.precision.upper()}-{args.recon}", "sample": sample},
        "cpu_baseline": {"value": r["value"], "unit": "site-updates/s", "cores": r["cores"], "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": r["value"], "unit": "site-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---- one process per GPU: the only cross-rank traffic is the barrier and a max of the timings ----
class Ranks:
    """Replicas only: N independent lattices, no data-path collective."""

    def __init__(self, backend: str = "nccl", device=None):
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        self.device = device
        self.dist = None
        if self.world > 1:
            import torch.distributed as dist
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            kw = {"device_id": device} if (backend == "nccl" and device is not None) else {}
            dist.init_process_group(backend, rank=self.rank, world_size=self.world, **kw)
            self.dist = dist

    def barrier(self):
        if self.dist:
            self.dist.barrier()

    def max_over_ranks(self, x: float) -> float:
        if not self.dist:
            return float(x)
        import torch
        t = torch.tensor([x], dtype=torch.float64, device=self.device if self.device is not None else "cpu")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def whole_job_value(self, units_per_rank: float, seconds_local: float) -> float:
        """units all ranks processed / slowest rank's time (every rank does the same amount of work)."""
        return self.world * units_per_rank / self.max_over_ranks(seconds_local)

    def close(self):
        if self.dist:
            self.dist.destroy_process_group()


# ---- t-shards: one lattice over N GPUs (strong scaling) ---------------------------
def run_sharded(args):
    """`--shard-t`: rank k holds the k-th slab of time-slices of ONE lattice; the half-sweep kernel of a rank reads and
    writes the boundary links in its neighbour's store in place through a CUDA IPC mapping (NVLink), torch.distributed
    (NCCL) carries only the stream-ordered barrier after each half-sweep and the sum of 2 Nt slice sums per check."""
    import torch
    from paper_1212_5221_b200 import build as _build
    _build.build()
    from paper_1212_5221_b200 import gf, shards

    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    ranks = Ranks("nccl", dev)
    world, rank = ranks.world, ranks.rank
    dims = tuple(int(x) for x in args.lattice.split(","))
    Nx, Ny, Nz, Nt = dims
    V, S = Nx * Ny * Nz * Nt, args.sweeps_per_step
    peak, peak_src = peaks()
    tile = make_tile()
    stream = torch.cuda.Stream(device=dev)
    prec, recon = args.precision, args.recon
    reunit = 100 if prec != "dp" else 0

    class _Dist:      # the part of torch.distributed the shard helpers use, also for a single rank
        def __init__(self, d):
            self.d = d

        def get_world_size(self):
            return world

        def get_rank(self):
            return rank

        def __getattr__(self, n):
            return getattr(self.d, n)

    fx, comm, (t0, nloc) = shards.make_rank_shard(_Dist(ranks.dist), dev, stream, Nx, Ny, Nz, Nt,
                                                   precision=PREC_NAMES[prec], recon=recon)
    reps = reps_for((Nx, Ny, Nz, nloc))
    with torch.cuda.stream(stream):
        slab = torch.from_numpy(tile).to(dev).repeat(*reps, 1, 1, 1, 1).contiguous()
    stream.synchronize()
    fx.set_links(slab)
    del slab

    def step():
        return fx.run(LANDAU, OR, OMEGA, seed=7, max_sweeps=S, eps=-1.0, check_every=S, reunit_every=reunit)

    for _ in range(args.warmup):
        step()
    sampler = ClockSampler(local)
    ranks.barrier(); torch.cuda.synchronize()
    sampler.start()
    gf.gf_launch_count(fx.ctx, reset=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        r = step()
    e1.record(stream)
    ranks.barrier(); torch.cuda.synchronize()
    ms = ranks.max_over_ranks(e0.elapsed_time(e1))
    launches = gf.gf_launch_count(fx.ctx, reset=True)
    clocks = sampler.stop()
    bpsu = bytes_per_site_update(prec, recon)
    # every rank streams its own slab once per half-sweep: aggregate algorithmic bytes over the slowest rank's time
    achieved = bpsu * V * S * args.steps / (ms * 1e-3) / 1e9 / world
    if rank == 0:
        line = {
            "metric": "site-updates/s (Landau OR sweep incl. F/theta reductions)", "value": V * S * args.steps / (ms * 1e-3),
            "unit": "site-updates/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": DTYPE_NAMES[prec], "data": "synthetic",
            "config": {"workload": f"Landau OR omega=1.7, {'x'.join(map(str, dims))} (BASELINE.json configs[4]), "
                                   f"{prec.upper()}-{recon}, ONE lattice split along t over {world} GPU(s)",
                       "lattice": list(dims), "precision": prec, "recon": recon,
                       "parallelism": f"t-shards x{world}: {Nt // world} slices per GPU, boundary links read and written in "
                                      "place in the neighbour's store (CUDA IPC mapping over NVLink), NCCL for the barrier "
                                      "per half-sweep and the slice sums per check",
                       "l2": "every slab >> 126 MB L2: streams from HBM"},
            "paper_gflops": V * S * args.steps / (ms * 1e-3) * 2274 / 1e9,
            "gpu_launches": launches, "F": r["F"], "theta": r["theta"],
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": None, "kernel": "gf::sweep_kernel (one half-sweep, per GPU, whole step incl. barriers)",
                         "peak_source": peak_src, "bytes_per_site_update": bpsu},
            "clocks": clocks, "e2e": None, "cpu_baseline": None,
            "comm_calls": comm.calls if comm else {"barrier": 0, "allreduce": 0},
        }
        print(json.dumps(line), flush=True)
    fx.close()
    ranks.close()


# ---- the CUDA path ----------------------------------------------------------------------------
def run_ours(args):
    import torch
    from paper_1212_5221_b200 import build as _build
    _build.build()                          # in-tree libgf.so: a no-op when it is up to date (nvcc, sm_100a)
    from paper_1212_5221_b200 import gf     # fails loudly if libgf.so is missing

    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    ranks = Ranks("nccl", dev)
    world, rank = ranks.world, ranks.rank
    max_over_ranks = ranks.max_over_ranks

    def barrier():
        ranks.barrier()
        torch.cuda.synchronize()

    dims = tuple(int(x) for x in args.lattice.split(","))
    Nx, Ny, Nz, Nt = dims
    V = Nx * Ny * Nz * Nt
    S = args.sweeps_per_step
    peak, peak_src = peaks()
    lat_name = "x".join(map(str, dims))

    tile = make_tile()
    su2 = args.group == "su2"
    if su2:
        from paper_1212_5221_b200 import inputs
        args.recon, args.no_variants, args.no_cpu_baseline = 4, True, True
        head_tile = inputs.as_real(inputs.make_config_su2(*TILE, TILE_EPS, *TILE_SEEDS))
    else:
        head_tile = tile
    reps = reps_for(dims)
    stream = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(stream):
        tile_dev = torch.from_numpy(head_tile).to(dev)
        links_dev = tile_dev.repeat(*reps, 1, 1, 1, 1).contiguous()     # StandardPattern, f64, in HBM
    stream.synchronize()
    del tile_dev

    GAUGE = {"landau": 0, "coulomb": 1, "mag": 2}[args.gauge]
    ALGO = {"or": 0, "sr": 1, "sa": 2, "micro": 3}[args.algo]
    if (GAUGE, ALGO) != (LANDAU, OR):
        args.no_variants, args.no_cpu_baseline, args.no_others = True, True, True
    TRAFFIC_KEY = "or" if ALGO == OR and GAUGE == LANDAU else ("sa_mag" if (GAUGE, ALGO) == (2, 2) else ("sa" if (GAUGE, ALGO) == (0, 2) else "none"))

    def bench_one(prec: str, recon: int, steps: int, warmup: int, e2e: bool, sample_clocks: bool):
        reunit = 100 if prec != "dp" else 0
        if ALGO != OR and recon == 12:
            reunit = 16          # heatbath / microcanonical sweeps on 12-real storage
        out = {}
        with gf.GaugeFixer(Nx, Ny, Nz, Nt, precision=PREC_NAMES[prec], recon=18 if su2 else recon, cuda_stream=stream,
                           su2=su2) as fx:
            if args.block:
                gf.gf_debug_set_block(fx.ctx, args.block)
            fx.set_links(links_dev)

            def step():
                return fx.run(GAUGE, ALGO, args.param, seed=7, max_sweeps=S, eps=-1.0, check_every=S, reunit_every=reunit)

            for _ in range(warmup):
                step()
            sampler = ClockSampler(local) if sample_clocks else None
            barrier()
            if sampler:
                sampler.start()
            gf.gf_launch_count(fx.ctx, reset=True)
            gf.gf_kernel_timing(fx.ctx, True)
            gf.gf_kernel_time_ms(fx.ctx, reset=True)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(steps):
                r = step()
            e1.record(stream)
            barrier()
            ms = max_over_ranks(e0.elapsed_time(e1))
            kern_ms, kern_n = gf.gf_kernel_time_ms(fx.ctx, reset=True)
            gf.gf_kernel_timing(fx.ctx, False)
            launches = gf.gf_launch_count(fx.ctx, reset=True)
            if sampler:
                out["clocks"] = sampler.stop()
            bpsu = bytes_per_site_update(prec, recon, 3 if GAUGE == 1 else 4)
            per_launch_bytes = bpsu * (V // 2)
            achieved = per_launch_bytes / (kern_ms / kern_n * 1e-3) / 1e9
            out.update({
                "precision": prec, "recon": recon, "steps": steps, "ms_per_step": ms / steps,
                "value": world * V * S * steps / (ms * 1e-3),
                "paper_gflops": world * V * S * steps / (ms * 1e-3) * 2274 / 1e9,
                "gpu_launches": launches, "F": r["F"], "theta": r["theta"],
                "kernel_share_of_step": kern_ms / ms,
                "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                             "frac": achieved / peak, "frac_of_8TBps_nominal": achieved / 8000.0,
                             "traffic": NCU_TRAFFIC.get((TRAFFIC_KEY, prec, recon, lat_name)),
                             "traffic_source": f"profiles/traffic.csv, ncu --set full capture of the kernels of commit {NCU_TRAFFIC_COMMIT}",
                             "kernel": "gf::sweep_su2_kernel (one half-sweep)" if su2 else "gf::sweep_kernel (one half-sweep)",
                             "peak_source": peak_src,
                             "algorithmic_bytes_per_launch": per_launch_bytes,
                             "bytes_per_site_update": bpsu, "avg_launch_ms": kern_ms / kern_n,
                             "launches_timed": kern_n},
            })
            if e2e:
                eb = 8 if prec == "dp" else 4
                tdt = torch.float64 if prec == "dp" else torch.float32
                nbytes = V * (32 if su2 else 72) * eb
                import psutil
                need = 2 * nbytes * max(1, world)
                if psutil.virtual_memory().available < 1.15 * need:
                    out["e2e"] = {"value": None, "unit": "site-updates/s", "h2d_bytes_per_step": nbytes,
                                  "d2h_bytes_per_step": nbytes, "skipped": "not enough host memory for pinned buffers"}
                else:
                    h_in = torch.empty(links_dev.shape, dtype=tdt, pin_memory=True)
                    h_out = torch.empty(links_dev.shape, dtype=tdt, pin_memory=True)
                    with torch.cuda.stream(stream):
                        h_in.copy_(links_dev.to(tdt) if tdt != links_dev.dtype else links_dev)
                    stream.synchronize()

                    def e2e_step():
                        fx.set_links(h_in)                          # host -> device (+ layout conversion)
                        rr = step()                                 # S sweeps + F/theta
                        fx.get_links(out=h_out)                     # device -> host
                        return rr

                    e2e_step()
                    n_e2e = max(1, steps // 2)
                    barrier()
                    t0 = time.perf_counter()
                    for _ in range(n_e2e):
                        rr = e2e_step()
                    barrier()
                    sec = max_over_ranks(time.perf_counter() - t0)
                    out["e2e"] = {"value": world * V * S * n_e2e / sec, "unit": "site-updates/s",
                                  "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes + 24,
                                  "steps": n_e2e, "ms_per_step": 1e3 * sec / n_e2e,
                                  "timing": "host wall clock around gf_set_links(host) + gf_run + gf_get_links(host), "
                                            "each synchronous; max over ranks"}
                    del h_in, h_out
        return out

    head = bench_one(args.precision, args.recon, args.steps, args.warmup, not args.no_e2e, True)
    variants = []
    if not args.no_variants:
        for prec, recon in (("sp", 18), ("sp", 12), ("dp", 12), ("mp", 12)):
            if (prec, recon) == (args.precision, args.recon):
                continue
            v = bench_one(prec, recon, max(1, min(2, args.steps)), 1, False, False)
            variants.append({"precision": prec, "recon": recon, "dtype": DTYPE_NAMES[prec],
                             "value": v["value"], "ms_per_step": v["ms_per_step"], "steps": v["steps"],
                             "roofline_achieved_gbs": v["roofline"]["achieved"], "roofline_frac": v["roofline"]["frac"],
                             "bytes_per_site_update": v["roofline"]["bytes_per_site_update"],
                             "kernel_share_of_step": v["kernel_share_of_step"]})

    def bench_other(dims_o, gauge, prec, recon, copies, sweeps, label, su2=False, track=False, algo=OR, param=OMEGA, key=None):
        """Side measurement (not the headline): `sweeps` OR sweeps of `copies` lattices of extent dims_o.
        key: the name under which the measurement also enters the compact `roofline.modes` summary."""
        ox, oy, oz, ot = dims_o
        Vo = ox * oy * oz * ot
        nd = 3 if gauge == 1 else 4
        r_o = (ot // TILE[3], ox // TILE[0], oy // TILE[1], oz // TILE[2])
        if su2:
            from paper_1212_5221_b200 import inputs
            recon = 4            # reals kept per SU(2) link (first row of the matrix)
            src_tile = inputs.as_real(inputs.make_config_su2(*TILE, TILE_EPS, *TILE_SEEDS))
        else:
            src_tile = tile
        with torch.cuda.stream(stream):
            src = torch.from_numpy(src_tile).to(dev).repeat(*r_o, 1, 1, 1, 1).contiguous()
        with gf.GaugeFixer(ox, oy, oz, ot, precision=PREC_NAMES[prec], recon=18 if su2 else recon, n_copies=copies,
                           cuda_stream=stream, su2=su2, track_transform=track) as fx:
            fx.set_links(src)
            del src
            # heatbath / microcanonical sweeps on 12-real storage need frequent reprojection
            ru = 16 if (algo != OR and recon == 12) else 0
            fx.run_batch(gauge, algo, param, seed=7, max_sweeps=10, eps=-1.0, check_every=10, reunit_every=ru)
            # pass 1: the run as a user makes it (no events between the launches: back-to-back half-sweeps with
            # programmatic dependent launch) -> value;  pass 2: events around every half-sweep -> roofline
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            fx.run_batch(gauge, algo, param, seed=7, max_sweeps=sweeps, eps=-1.0, check_every=sweeps, reunit_every=ru)
            e1.record(stream)
            stream.synchronize()
            ms = e0.elapsed_time(e1)
            gf.gf_kernel_timing(fx.ctx, True)
            gf.gf_kernel_time_ms(fx.ctx, reset=True)
            fx.run_batch(gauge, algo, param, seed=7, max_sweeps=sweeps, eps=-1.0, check_every=sweeps, reunit_every=ru)
            kern_ms, kern_n = gf.gf_kernel_time_ms(fx.ctx, reset=True)
            gf.gf_kernel_timing(fx.ctx, False)
        bpsu = bytes_per_site_update(prec, recon, nd)
        if track:       # g(x) (18 reals, 4 for SU(2)) read and written once per site update
            bpsu += 2 * (4 if su2 else 18) * (8 if prec == "dp" else 4)
        ach = bpsu * (copies * Vo // 2) / (kern_ms / kern_n * 1e-3) / 1e9
        eff = bpsu * copies * Vo * sweeps / (ms * 1e-3) / 1e9        # whole run incl. gaps, reductions, reprojection
        store = copies * Vo * 4 * recon * (8 if prec == "dp" else 4)
        return {"workload": label, "key": key, "gauge_group": "SU(2)" if su2 else "SU(3)", "lattice": list(dims_o), "copies": copies, "precision": prec, "recon": recon,
                "sweeps": sweeps, "value": copies * Vo * sweeps / (ms * 1e-3), "unit": "site-updates/s",
                "avg_launch_ms": kern_ms / kern_n, "roofline_achieved_gbs": ach, "roofline_frac": ach / peak,
                "whole_run_gbs": eff, "whole_run_frac": eff / peak,
                "bytes_per_site_update": bpsu, "link_store_bytes": store,
                "resident_in": "L2 (126 MB): not an HBM measurement" if store < 100e6 else "HBM"}

    def bench_shards_one_device(dims_o, prec, recon, n_shards, sweeps, label):
        """Side measurement: ONE lattice as n_shards t-shards on this device, all on one stream, every shard driven by its
        own host thread (thread communicator).  Shows what the in-place boundary access and the per-half-sweep ordering
        cost against the unsharded run of the same lattice (the multi-GPU path itself needs several GPUs)."""
        import threading
        from paper_1212_5221_b200 import shards
        ox, oy, oz, ot = dims_o
        Vo = ox * oy * oz * ot
        parts = shards.partition_t(ot, n_shards)
        fxs = [gf.GaugeFixer(ox, oy, oz, n, precision=PREC_NAMES[prec], recon=recon, cuda_stream=stream, shard=(t0, ot))
               for t0, n in parts]
        comms = shards.ThreadComm.group(n_shards)
        res = {}
        try:
            for k, fx in enumerate(fxs):
                fx.attach(fxs[(k - 1) % n_shards], fxs[(k + 1) % n_shards])
                fx.set_comm(comms[k].comm)

            def work(k):
                t0, n = parts[k]
                with torch.cuda.stream(stream):
                    src = torch.from_numpy(tile).to(dev).repeat(n // TILE[3], ox // TILE[0], oy // TILE[1], oz // TILE[2], 1, 1, 1, 1).contiguous()
                stream.synchronize()
                fxs[k].set_links(src)
                del src
                fxs[k].run(LANDAU, OR, OMEGA, seed=7, max_sweeps=4, eps=-1.0, check_every=4)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                comms[k].shared.barrier.wait()
                if k == 0:
                    e0.record(stream)
                r = fxs[k].run(LANDAU, OR, OMEGA, seed=7, max_sweeps=sweeps, eps=-1.0, check_every=sweeps)
                comms[k].shared.barrier.wait()
                if k == 0:
                    e1.record(stream)
                    stream.synchronize()
                    res["ms"], res["F"] = e0.elapsed_time(e1), r["F"]

            th = [threading.Thread(target=work, args=(k,)) for k in range(n_shards)]
            for t in th:
                t.start()
            for t in th:
                t.join()
        finally:
            for fx in fxs:
                fx.close()
        bpsu = bytes_per_site_update(prec, recon)
        eff = bpsu * Vo * sweeps / (res["ms"] * 1e-3) / 1e9
        return {"workload": label, "gauge_group": "SU(3)", "lattice": list(dims_o), "copies": 1, "shards": n_shards,
                "precision": prec, "recon": recon, "sweeps": sweeps, "value": Vo * sweeps / (res["ms"] * 1e-3),
                "unit": "site-updates/s", "whole_run_gbs": eff, "whole_run_frac": eff / peak, "bytes_per_site_update": bpsu,
                "F": res["F"], "resident_in": "HBM"}

    others = []
    if rank == 0 and world == 1 and not args.no_others:
        del links_dev
        links_dev = None
        torch.cuda.empty_cache()
        others = [
            bench_other((32, 32, 32, 64), 0, "dp", 18, 1, 200, "Landau OR, 32^3x64, DP-18", key="dp18_32x32x32x64"),
            bench_other((32, 32, 32, 64), 0, "sp", 12, 1, 200, "Landau OR, 32^3x64, SP-12", key="sp12_32x32x32x64"),
            bench_other((32, 32, 32, 64), 1, "sp", 12, 1, 200, "Coulomb OR, 32^3x64, SP-12 (BASELINE.json configs[2])", key="coulomb_sp12_32x32x32x64"),
            bench_other((16, 16, 16, 16), 0, "dp", 18, 1, 1000, "Landau OR, 16^4, DP-18, one copy (configs[1])"),
            bench_other((16, 16, 16, 16), 0, "dp", 18, 64, 100, "Landau OR, 64 gauge copies of 16^4 per launch, DP-18"),
            bench_other((32, 32, 32, 32), 0, "sp", 12, 16, 100, "Landau OR, 16 gauge copies of 32^4 per launch, SP-12"),
            bench_other((64, 64, 64, 256), 0, "sp", 12, 1, 50, "Landau OR, 64^3x256, SP-12, accumulating g(x) (a8)", track=True),
            bench_other((64, 64, 64, 256), 2, "dp", 18, 1, 30, "MAG OR, 64^3x256, DP-18", key="mag_dp18"),
            bench_other((64, 64, 64, 256), 0, "sp", 12, 1, 30, "Landau simulated-annealing heatbath T=1 (Philox), 64^3x256, SP-12", algo=2, param=1.0, key="sa_sp12"),
            bench_other((64, 64, 64, 256), 0, "dp", 18, 1, 20, "Landau simulated-annealing heatbath T=1 (Philox), 64^3x256, DP-18", algo=2, param=1.0, key="sa_dp18"),
            bench_other((64, 64, 64, 256), 0, "mp", 12, 1, 20, "Landau simulated-annealing heatbath T=1 (Philox), 64^3x256, MP-12", algo=2, param=1.0, key="sa_mp12"),
            bench_other((64, 64, 64, 256), 2, "dp", 18, 1, 20, "MAG simulated-annealing heatbath T=0.5 (Philox), 64^3x256, DP-18", algo=2, param=0.5, key="sa_mag_dp18"),
            bench_other((64, 64, 64, 256), 0, "sp", 12, 1, 30, "Landau stochastic relaxation p=0.5 (Philox), 64^3x256, SP-12", algo=1, param=0.5, key="sr_sp12"),
            bench_other((64, 64, 64, 256), 0, "sp", 4, 1, 100, "SU(2) Landau OR, 64^3x256, SP (4 reals per link)", su2=True, key="su2_sp"),
            bench_other((64, 64, 64, 256), 0, "dp", 4, 1, 100, "SU(2) Landau OR, 64^3x256, DP (4 reals per link)", su2=True, key="su2_dp"),
            bench_other((64, 64, 64, 256), 2, "mp", 4, 1, 100, "SU(2) MAG OR, 64^3x256, MP", su2=True),
            bench_shards_one_device((64, 64, 64, 256), "sp", 12, 4, 50,
                                    "Landau OR, 64^3x256, SP-12, ONE lattice as 4 t-shards on one device (one stream)"),
        ]

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        links_dev = None
        torch.cuda.empty_cache()
        r = oracle_leg(tile, args.precision, 20, 5, 1)
        cpu = {"value": r["value"], "unit": "site-updates/s", "cores": r["cores"], "kind": "oracle",
               "sample": f"5 x 20 Landau OR sweeps + F/theta of oracle/gf_oracle.cpp ({args.precision.upper()}) on a "
                         f"{'x'.join(map(str, ORACLE_SAMPLE_DIMS))} sample (V={r['V']}) of the workload, "
                         f"{r['seconds']:.1f} s"}

    if rank == 0:
        # compact per-mode summary inside `roofline` (the driver's record keeps that object): per-kernel fraction of
        # roofline.peak (CUDA events around every half-sweep) and whole-run G site-updates/s; 64^3x256 unless the key
        # names another lattice; sa_* = simulated-annealing heatbath, sr_* = stochastic relaxation half-sweeps
        modes = {f"{args.precision}{args.recon}": [round(head["roofline"]["frac"], 4), round(head["value"] / world / 1e9, 3)]}
        for v in variants:
            modes[f"{v['precision']}{v['recon']}"] = [round(v["roofline_frac"], 4), round(v["value"] / world / 1e9, 3)]
        for o in others:
            if o.get("key"):
                modes[o["key"]] = [round(o["roofline_frac"], 4), round(o["value"] / 1e9, 3)]
        head["roofline"]["modes"] = modes
        head["roofline"]["modes_columns"] = ["kernel_frac_of_peak", "G_site_updates_per_s_per_gpu"]
        line = {
            "metric": "site-updates/s (Landau OR sweep incl. F/theta reductions)", "value": head["value"],
            "unit": "site-updates/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": DTYPE_NAMES[args.precision], "data": "synthetic",
            "config": {"workload": f"{'SU(2) ' if su2 else ''}{'Landau OR omega=1.7' if (GAUGE, ALGO, args.param) == (LANDAU, OR, OMEGA) else f'{args.gauge.capitalize()} {args.algo.upper()} param={args.param:g} (side study)'}, {lat_name} (BASELINE.json configs[4]), "
                                   f"{args.precision.upper()}-{args.recon}, one lattice per GPU",
                       "lattice": list(dims), "precision": args.precision, "recon": args.recon,
                       "step": f"{S} sweeps (= {2 * S} half-sweep kernels) + "
                               f"{'DP reunitarisation + ' if args.precision != 'dp' else ''}one F/theta reduction",
                       "l2": "link store %.1f GB >> 126 MB L2: every half-sweep streams from HBM, no flush needed"
                             % (V * 4 * args.recon * (8 if args.precision == 'dp' else 4) / 1e9),
                       "parallelism": ("replicas only" if world > 1 else "single GPU") +
                                      " (--shard-t instead splits ONE lattice along t over the ranks: DESIGN.md §10, unmeasured on more than one GPU)"},
            "paper_gflops": head["paper_gflops"],
            "paper_context": "3.5 TFlops on 16 Tesla C2070, 64^3x256 SP (PAPER.md:518); other hardware, context only",
            "gpu_launches": head["gpu_launches"], "F": head["F"], "theta": head["theta"],
            "kernel_share_of_step": head["kernel_share_of_step"],
            "roofline": head["roofline"], "clocks": head.get("clocks"),
            "e2e": head.get("e2e"), "cpu_baseline": cpu, "variants": variants,
            "other_workloads": others,
        }
        print(json.dumps(line), flush=True)
    ranks.close()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.shard_t:
        run_sharded(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
