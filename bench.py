#!/usr/bin/env python
"""bench.py -- throughput of the Metropolis colour sweep on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c4]

One "step" is one pass of the whole hot path over the resident lattice: the workload's sweeps
(config 4: its 200 timed sweeps; one kernel per colour per sweep: SURVEY 8(a) rows a4, a6) and one
M/E measurement (row a5; for the sc engine it is reduced inside the last sweep's kernels).  Lattice build, colouring and the initial state (rows a1-a3)
are set-up, done once before the warm-up.

Workload at N = 1: config 4 of BASELINE.json, simple cubic L = 464 (99,897,344 spins, 1.2 GB
of fp32 SoA state, far larger than the 126 MB L2, so no flush between iterations), J = 1,
K = 0.01 along z, random start from seed 1, T = 1.44.  With N > 1 every rank runs an
independent replica of that workload (seed + rank): the path has no multi-GPU exchange in
scope ("replicas only"), so scaling is weak and there is no collective
on the data path.

After the headline's timed region the default run (c4, N = 1) also times the other configs and the size sweep of the paper's
Fig. 2 for about a second each (`workloads`), repeats the timed region twice more (`repeats`) and times the same sweeps with a
measurement after every one (`with_per_sweep_measurement`); `roofline.cycles_per_launch` / `updates_per_clock` are the
clock-independent figures ("report for every timed config").

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle instead (the tier's
reference arm): single-threaded, on a bounded sample of the same workload.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

# Sweeps of one step: config 4 is specified as "200 timed sweeps" (BASELINE.json), so its step is those 200 sweeps
# followed by the measurement; the secondary workloads (scans of hundreds to thousands of sweeps per temperature)
# use 50-100.
SWEEPS_BY_WORKLOAD = {"c4": 200, "c1": 100, "c2": 100, "c3": 50, "c5": 50, "x_bcc256": 50, "x_fcc256": 20}
SWEEPS_PER_STEP = 10
METRIC = "attempted spin updates/sec (Gupd/s) and % of HBM roofline, 1 B200"
UNIT = "Gupd/s"

# DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of ONE launch of the dominant kernel,
# from the `ncu --set full` capture summarised in profiles/ (file named beside each value).
NCU_TRAFFIC_BYTES_PER_LAUNCH = {}
try:
    with open(os.path.join(ROOT, "profiles", "traffic.csv")) as _f:
        for _ln in _f:
            if _ln.strip() and not _ln.startswith("#"):
                _k, _v = _ln.split(",")[:2]
                NCU_TRAFFIC_BYTES_PER_LAUNCH[_k.strip()] = float(_v)
except OSError:
    pass


def algorithmic_bytes_per_update(cfg, n_colours):
    """SURVEY 8(d) / DESIGN.md section 7: what one colour pass must move, per attempted update."""
    if cfg["kind"] in ("sc", "bcc"):
        return 36.0      # read own 12 B + the other colour once 12 B + write own 12 B
    if cfg["kind"] == "fcc":
        return 60.0      # own 12 + three other sublattices 36 + write 12
    # table engine (ELL, maxdeg 12): table 48 + site id 4 + (K_i, e_i) 16 + own float4 16 read + 16 written;
    # the gathered neighbour spins (58 MB in all) are L2 traffic
    return 100.0


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.FIELDS,
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
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
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.f:
            c = [x.strip() for x in ln.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for name, v in zip(names, c[3:7]):
                if v == "Active":
                    reasons.add(name)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


def reduce_over_ranks(maxima, sums, device):
    """The only cross-rank step of the bench (replicas only: no data-path collective): every timing
    is the MAX over ranks, every count the SUM.  `device` is where the tensors live ("cuda:k" under
    NCCL, "cpu" under gloo in the CPU tests).  World size 1 (no process group) returns the inputs."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(x) for x in maxima], [int(x) for x in sums]
    t = torch.tensor([float(x) for x in maxima], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor([int(x) for x in sums] + [0], device=device, dtype=torch.int64)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.tolist()], [int(x) for x in c.tolist()[:-1]]


def replica_seed(cfg, rank):
    """Rank r runs an independent replica of the workload: same lattice and parameters, seed + r."""
    return int(cfg["seed"]) + int(rank)


def make_context(cfg, seed_offset, device):
    import paper_2106_11286_b200 as hb
    if cfg["kind"] == "sphere":
        lat = hb.Lattice.fcc_sphere(cfg["R"], cfg["K"], cfg["e"], cfg["K_surf"], cfg.get("colouring", "greedy"))
    else:
        lat = hb.Lattice(cfg["kind"], cfg["L"])
    ctx = hb.Context(lat, cfg["J"], cfg["K"], cfg["e"], replica_seed(cfg, seed_offset), device=device)
    if cfg["start"] == "random":
        ctx.init_random()
    else:
        ctx.init_aligned(cfg["e"])
    return ctx


def host_cpu():
    """Model string and core count of the box the oracle is timed on ("oracle timing beside it")."""
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as f:
            for ln in f:
                if ln.lower().startswith("model name"):
                    model = ln.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    return model, os.cpu_count() or 0


def sample_lattice_label(scfg):
    return "%s %s" % (scfg["kind"], scfg.get("L", scfg.get("R")))


def cpu_sample_cfg(cfg):
    """A bounded sample of the workload for the single-threaded oracle (about 10-30 s of CPU work)."""
    if cfg["kind"] == "sc" and cfg["L"] > 232:
        return dict(cfg, L=232), "sc L=232 (1/8 of the L=464 volume), same J, K, e, T, random start"
    if cfg["kind"] == "fcc" and cfg["L"] > 64:
        return dict(cfg, L=64), "fcc L=64 (1/8 of the volume), same parameters"
    if cfg["kind"] == "sphere" and cfg["R"] > 30:
        return dict(cfg, R=30), "fcc sphere R=30 (1/8 of the volume), same parameters"
    return dict(cfg), "the full workload"


def make_oracle_state(cfg):
    import oracle
    if cfg["kind"] == "sphere":
        lat = oracle.Lattice.fcc_sphere(cfg["R"], cfg["K"], cfg["e"], cfg["K_surf"], cfg.get("colouring", "greedy"))
    else:
        lat = getattr(oracle.Lattice, cfg["kind"])(cfg["L"])
        lat.set_uniform_anisotropy(cfg["K"], cfg["e"])
    st = oracle.State32(lat, cfg["J"], cfg["seed"])
    if cfg["start"] == "random":
        st.init_random()
    else:
        st.init_aligned(cfg["e"])
    return lat, st


def run_cpu_baseline(cfg, budget_attempts=2.5e8):   # ~14 s at the oracle's 55 ns per attempt
    scfg, what = cpu_sample_cfg(cfg)
    lat, st = make_oracle_state(scfg)
    T = scfg["T"][0]
    n = lat.n
    sweeps = max(1, int(round(budget_attempts / n)))
    st.sweep(T, 1)
    t0 = time.perf_counter()
    st.sweep(T, sweeps)
    st.measure()
    dt = time.perf_counter() - t0
    model, nproc = host_cpu()
    return {"value": n * sweeps / dt / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": "%s; %d sweeps + 1 measurement (%d attempts), O32 single thread" % (what, sweeps, n * sweeps),
            "sample_lattice": sample_lattice_label(scfg), "cpu_model": model, "nproc": nproc,
            "ns_per_update": dt / (n * sweeps) * 1e9}



def timed_rate(ctx, T, seconds, sweep=None):
    """Attempted updates per second of ctx.sweep (or `sweep`, a callable taking a sweep count) in a run sized for about `seconds`,
    timed with CUDA events on the context's stream after a warm-up; returns (updates per second, sweeps, ms)."""
    import torch
    sweep = sweep or (lambda k: ctx.sweep(T, k))
    sweep(16)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(); sweep(16); b.record(); torch.cuda.synchronize()
    per_sweep_ms = max(a.elapsed_time(b) / 16, 1e-4)
    k = int(min(max(16, seconds * 1e3 / per_sweep_ms), 200000))
    k -= k % 8                                   # whole replayed graphs of 8 sweeps
    a.record(); sweep(k); b.record(); torch.cuda.synchronize()
    ms = a.elapsed_time(b)
    return float(ctx.n) * ctx.n_replicas * k / (ms * 1e-3), k, ms


def run_secondary_workloads(device, local, peak, alu_peak, seconds=1.0):
    """SURVEY 8(d), "report for every timed config": after the headline's timed region the default run also times c1 (one
    system, and 1184 replicas in one context), c2, c3, c5 (greedy and parity colouring) for about a second each and the
    size sweep of Fig. 2 [P:44,48] for a third of a second per size, device-resident, CUDA events, clocks sampled per
    workload.  Rates of whole hb_sweep calls (all colours, launch gaps included): these are the driver's numbers for the
    configs that are not the headline."""
    import paper_2106_11286_b200 as hb
    from paper_2106_11286_b200 import workloads
    out = {}

    def one(name, cfg, ctx, secs, extra=None):
        T = cfg["T"][0]
        sampler = ClockSampler(local)
        time.sleep(0.3)
        s0 = ctx.stats()
        rate, k, ms = timed_rate(ctx, T, secs)
        ctx.measure()
        s1 = ctx.stats()
        clocks = sampler.stop()
        _, n_colours = ctx.colouring()
        bpu = algorithmic_bytes_per_update(cfg, n_colours)
        kernel = {"sc": "k_sweep_sc", "bcc": "k_sweep_bravais", "fcc": "k_sweep_bravais", "sphere": "k_sweep_ell"}[cfg["kind"]]
        if cfg["kind"] == "sc" and ctx.n_replicas > 1:
            kernel = "k_sweeps_sc_coop (one block per replica)"
        elif cfg["kind"] == "sc" and ctx.get_option("sc_kernel") >= 1:
            kernel = "k_sweep_sc_ws"
        elif cfg["kind"] == "sc" and ctx.n <= 8192:
            kernel = "k_sweeps_sc_coop (one block)"
        elif cfg["kind"] in ("bcc", "fcc") and ctx.get_option("br_kernel") >= 1:
            kernel = "k_sweep_bravais_ws"
        rec = {"value": rate / 1e9, "unit": UNIT, "n_spins": ctx.n * ctx.n_replicas, "colours": n_colours, "T": T, "sweeps": k,
               "ms_per_sweep": ms / k, "kernel": kernel,
               "roofline": {"hbm": bpu * rate / 1e9 / peak, "alu": rate / 1e9 / alu_peak, "algorithmic_bytes_per_update": bpu,
                            "l2_resident": 12.0 * ctx.n * ctx.n_replicas <= 126e6},
               "acceptance_rate": (s1[1] - s0[1]) / max(1, s1[0] - s0[0]),
               "clocks": {"sm_mhz": clocks["sm_mhz"], "reasons": clocks["reasons"]}}
        if clocks["sm_mhz"]:
            rec["updates_per_clock"] = rate / (clocks["sm_mhz"] * 1e6)
        rec.update(extra or {})
        out[name] = rec
        ctx.close()

    C = workloads.CONFIGS
    one("c1", C["c1"], make_context(C["c1"], 0, device), seconds)
    c1r = hb.Context(hb.Lattice("sc", 16, n_replicas=1184), C["c1"]["J"], C["c1"]["K"], C["c1"]["e"], C["c1"]["seed"], device=device)
    c1r.init_random()
    one("c1_x1184_replicas", C["c1"], c1r, seconds, {"replicas": 1184})
    one("c2", C["c2"], make_context(C["c2"], 0, device), seconds)
    one("c3", C["c3"], make_context(C["c3"], 0, device), seconds)
    one("c5", C["c5"], make_context(C["c5"], 0, device), seconds, {"colouring": "greedy first-fit"})
    c5p = dict(C["c5"], colouring="parity")
    one("c5_parity", c5p, make_context(c5p, 0, device), seconds, {"colouring": "the four parity classes"})
    sizes = {}
    for L in (16, 32, 64, 96, 128, 192, 256, 320, 384, 464):
        cfg = dict(C["c4"], L=L)
        ctx = make_context(cfg, 0, device)
        rate, k, ms = timed_rate(ctx, cfg["T"][0], seconds / 3)
        sizes[str(L)] = {"value": rate / 1e9, "ns_per_update": 1e9 / rate, "sweeps": k}
        ctx.close()
    out["size_sweep_sc"] = {"unit": UNIT, "T": C["c4"]["T"][0], "K": C["c4"]["K"], "by_L": sizes,
                            "note": "the shape of the paper's Fig. 2 [P:44,48]: rate against lattice size, one system per run"}
    return out

def run_reference(args, cfg, name):
    """--impl reference: the CPU oracle as it stands, one sweep of the bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    scfg, what = cpu_sample_cfg(cfg)
    lat, st = make_oracle_state(scfg)
    T = scfg["T"][0]
    for _ in range(args.warmup):
        st.sweep(T, 1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        st.sweep(T, 1)
        st.measure()
    dt = time.perf_counter() - t0
    value = lat.n * args.steps / dt / 1e9
    sample = "%s; each step = 1 sweep + 1 measurement of the sample, O32 single thread" % what
    model, nproc = host_cpu()
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        # the lattice that RAN: the bounded sample of the workload, not the workload's full size
        "config": {"workload": name,
                   "lattice": sample_lattice_label(scfg) if scfg == cfg else
                   "%s (bounded sample of the workload's %s)" % (sample_lattice_label(scfg), sample_lattice_label(cfg)),
                   "n_spins": lat.n, "T": T, "J": cfg["J"], "K": cfg["K"]},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                         "sample_lattice": sample_lattice_label(scfg), "cpu_model": model, "nproc": nproc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_slabs(args, cfg, rank, world, device, barrier):
    """--multi slabs: ONE lattice of the workload's size cut into `world` z-slabs (paper_2106_11286_b200.slabs.DistSlab):
    a step is the same SWEEPS_PER_STEP sweeps + one measurement of the WHOLE lattice; every colour pass is followed by the
    exchange of its two faces with the z-neighbours (NCCL send/recv; a single rank feeds its own ghost planes) and the
    measurement by one all_reduce of 4 doubles.  Timed on the device, MAX over ranks; total work is fixed: strong scaling."""
    import torch
    import torch.distributed as dist
    from paper_2106_11286_b200 import slabs
    if cfg["kind"] != "sc":
        raise SystemExit("--multi slabs: simple cubic workloads (c1, c4)")
    L = cfg["L"]
    Lx, Ly, Lz = (L, L, L) if isinstance(L, int) else L
    options = dict((kv.split("=", 1)[0], int(kv.split("=", 1)[1])) for kv in args.option)
    sl = slabs.DistSlab(Lx, Ly, Lz, cfg["J"], cfg["K"], cfg["e"], cfg["seed"], device=device, options=options,
                        peer_stores=args.slab_exchange in ("peer", "flags"), flags=args.slab_exchange == "flags")
    sl.init_random() if cfg["start"] == "random" else sl.init_aligned(cfg["e"])
    T = cfg["T"][0]
    for _ in range(args.warmup):
        sl.sweep(T, SWEEPS_PER_STEP)
        sl.measure()
    sampler = ClockSampler(int(device.split(":")[1])) if rank == 0 else None
    if sampler:
        time.sleep(0.5)
        sl.sweep(T, min(SWEEPS_PER_STEP, 20))
    l0, _ = sl.ctx.counters()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        sl.sweep(T, SWEEPS_PER_STEP)
        M, E = sl.measure()
    e1.record()
    barrier()
    l1, _ = sl.ctx.counters()
    clocks = sampler.stop() if sampler else None
    (ms,), (launches,) = reduce_over_ranks([e0.elapsed_time(e1)], [l1 - l0], device)
    if rank == 0:
        n = sl.n
        value = float(n) * SWEEPS_PER_STEP * args.steps / (ms * 1e-3) / 1e9
        peak, peak_src = measured_peaks()
        achieved = 36.0 * value     # GB/s: algorithmic 36 B per attempted update, copies and exchanges inside the time
        face_bytes = 2 * 2 * 3 * (Lx * Ly // 2) * 4   # per sweep and slab: 2 colours x 2 faces x 3 components, sent (and received)
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": args.workload, "lattice": "sc %s" % L, "n_spins": n, "colours": 2, "J": cfg["J"], "K": cfg["K"],
                       "T": T, "start": cfg["start"], "seed": cfg["seed"], "sweeps_per_step": SWEEPS_PER_STEP,
                       "measurements_per_step": 1, "options": options,
                       "multi_gpu": "slabs along z: %s planes per rank, %d bytes of boundary planes per rank and sweep (%s), "
                                    "one all_reduce of 32 bytes per measurement" % (
                                        [nz for _, nz in slabs.partition(Lz, world)], face_bytes,
                                        "stored by the colour kernels into the neighbours' ghost planes, neighbour flags inside the kernels"
                                        if sl.flags else ("stored by the colour kernels into the neighbours' ghost planes, a barrier per pass"
                                                          if sl.peer_stores else "sent as faces after every pass")),
                       "l2": "state %.0f MB per rank" % (12.0 * n / world / 1e6)},
            "ns_per_update": 1.0 / value, "clocks": clocks, "e2e": None, "gpu_launches": launches,
            "M": [float(x) for x in M], "E_per_spin": E / n,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak * world, "unit": "GB/s", "frac": achieved / (peak * world),
                         "traffic": None, "kernel": "k_sweep_sc_ws" if sl.ctx.get_option("sc_kernel") == 1 else "k_sweep_sc",
                         "peak_source": peak_src + " x n_gpus", "algorithmic_bytes_per_update": 36.0,
                         "note": "whole step (colour passes + face exchanges + measurement) against the aggregate peak"},
            "cpu_baseline": None}))
    sl.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4", help="c1..c5 (BASELINE.json configs); the headline is c4")
    ap.add_argument("--option", action="append", default=[], metavar="NAME=VALUE",
                    help="hb_set_option on the context (tuning knobs of DESIGN.md section 6), repeatable")
    ap.add_argument("--multi", default="replicas", choices=["replicas", "slabs"],
                    help="N > 1: independent replicas (default, weak scaling) or ONE lattice cut into z-slabs with a face "
                         "exchange per colour (strong scaling; simple cubic workloads; DESIGN.md section 9)")
    ap.add_argument("--slab-exchange", default="peer", choices=["peer", "flags", "copies"],
                    help="--multi slabs: boundary planes stored by the colour kernels straight into the neighbours' ghost planes "
                         "(peer memory, CUDA IPC between the ranks) with a one-word all_reduce as barrier between passes (peer, default) "
                         "or with neighbour flags set and awaited inside the kernels, boundary tiles first (flags; one GPU per rank), "
                         "or faces sent after every pass (copies: NCCL send/recv)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-workloads", action="store_true",
                    help="skip the block of secondary workloads (c1, c2, c3, c5, size sweep) the default c4 run adds after its timed region")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    from paper_2106_11286_b200 import workloads
    cfg = workloads.CONFIGS[args.workload]
    global SWEEPS_PER_STEP
    SWEEPS_PER_STEP = SWEEPS_BY_WORKLOAD.get(args.workload, SWEEPS_PER_STEP)
    if args.impl == "reference":
        return run_reference(args, cfg, args.workload)

    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    device = "cuda:%d" % local
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(device))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.multi == "slabs":
        return run_slabs(args, cfg, rank, world, device, barrier)

    ctx = make_context(cfg, rank, device)
    options = {}
    for kv in args.option:
        k, v = kv.split("=", 1)
        ctx.set_option(k, int(v))
        options[k] = int(v)
    T = cfg["T"][0]
    n = ctx.n
    _, n_colours = ctx.colouring()
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def timed_run(steps):
        """K steps; returns (region ms by CUDA events, ms inside hb_sweep only, kernel launches)."""
        l0, _ = ctx.counters()
        e0, e1 = ev(), ev()
        marks = []
        barrier()
        e0.record()
        for _ in range(steps):
            a, b = ev(), ev()
            a.record()
            ctx.sweep(T, SWEEPS_PER_STEP)
            b.record()
            ctx.measure()
            marks.append((a, b))
        e1.record()
        barrier()
        l1, _ = ctx.counters()
        return e0.elapsed_time(e1), sum(a.elapsed_time(b) for a, b in marks), l1 - l0

    for _ in range(args.warmup):
        ctx.sweep(T, SWEEPS_PER_STEP)
        ctx.measure()
    clocks = None
    for attempt in range(2):
        sampler = ClockSampler(local) if rank == 0 else None
        if sampler:
            time.sleep(0.5)          # nvidia-smi needs a moment before its first sample
            ctx.sweep(T, min(SWEEPS_PER_STEP, 20))   # keep the device under load while it starts
        stats0 = ctx.stats()
        ms, ms_sweeps, launches = timed_run(args.steps)
        stats1 = ctx.stats()
        clocks = sampler.stop() if sampler else None
        bad = clocks and any(r in clocks["reasons"] for r in ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"))
        if not bad:
            break
    (ms, ms_sweeps), (launches,) = reduce_over_ranks([ms, ms_sweeps], [launches], device)
    updates = float(n) * SWEEPS_PER_STEP * args.steps * world
    value = updates / (ms * 1e-3) / 1e9

    # best and median of >= 3 repeats of the timed region (the headline `value` is the FIRST region, the one
    # the contract describes), and the rate with a measurement after EVERY sweep (hb_sweep_series) beside the plain one
    repeat_values = [value]
    for _ in range(2):
        ms_r, _, _ = timed_run(args.steps)
        (ms_r,), _ = reduce_over_ranks([ms_r], [], device)
        repeat_values.append(updates / (ms_r * 1e-3) / 1e9)
    series_rate = None
    if world == 1 and ctx.n_replicas == 1:
        k_series = max(8, min(SWEEPS_PER_STEP, 64))
        ctx.sweep_series(T, 8)
        a, b = ev(), ev()
        a.record(); ctx.sweep_series(T, k_series); b.record(); torch.cuda.synchronize()
        series_rate = {"value": float(n) * k_series / (a.elapsed_time(b) * 1e-3) / 1e9, "unit": UNIT, "sweeps": k_series,
                       "what": "hb_sweep_series: M and E reduced after every sweep, kept on the device, one copy at the end"}

    # ---- end to end through the public API with HOST buffers ------------------------------------
    e2e = None
    if not args.no_e2e:
        host = [torch.empty(n, dtype=torch.float32).pin_memory() for _ in range(3)]
        ctx.get_spins(out=host)
        e2e_steps = max(1, args.steps)
        ctx.set_spins(*host); ctx.sweep(T, SWEEPS_PER_STEP); ctx.measure()
        barrier()
        t0 = time.perf_counter()
        # every step uploads its own input state from pinned host memory and reads its result back; the upload of step k+1
        # (hb_stage_spins, a stream of its own) runs while step k sweeps, hb_commit_spins makes it the state in stream order.
        # The first upload is exposed, and one more than the steps need is issued: both inside the timed region.
        ctx.stage_spins(*host)
        for _ in range(e2e_steps):
            ctx.commit_spins()                       # H2D of this step's input state has arrived: permute it into place
            ctx.stage_spins(*host)                   # H2D of the next step's input state, overlapping the sweeps below
            ctx.sweep(T, SWEEPS_PER_STEP)
            ctx.measure()                            # D2H of the step's result (M, E)
        ctx.commit_spins()
        barrier()
        dt = time.perf_counter() - t0
        (dt,), _ = reduce_over_ranks([dt], [], device)
        e2e = {"value": float(n) * SWEEPS_PER_STEP * e2e_steps * world / dt / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": 3 * n * 4, "d2h_bytes_per_step": 32, "steps": e2e_steps,
               "how": "hb_stage_spins / hb_commit_spins: the upload of step k+1 overlaps the sweeps of step k; steps + 1 uploads inside the timed region"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (one colour pass) -----------------------------------------
    peak, peak_src = measured_peaks()
    bytes_per_update = algorithmic_bytes_per_update(cfg, n_colours)
    launches_sweep = n_colours * SWEEPS_PER_STEP * args.steps
    avg_launch_s = ms_sweeps * 1e-3 / launches_sweep
    bytes_per_launch = bytes_per_update * n / n_colours
    achieved = bytes_per_launch / avg_launch_s / 1e9
    kernel = {"sc": "k_sweep_sc", "bcc": "k_sweep_bravais", "fcc": "k_sweep_bravais", "sphere": "k_sweep_ell"}[cfg["kind"]]
    if cfg["kind"] == "sc" and ctx.get_option("sc_kernel") >= 1:
        kernel = "k_sweep_sc_ws"
    if cfg["kind"] in ("bcc", "fcc") and ctx.get_option("br_kernel") >= 1:
        kernel = "k_sweep_bravais_ws"
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH.get(args.workload), "kernel": kernel, "peak_source": peak_src,
                "algorithmic_bytes_per_update": bytes_per_update, "bytes_per_launch": bytes_per_launch,
                "avg_launch_ms": avg_launch_s * 1e3, "frac_of_8TBs_nominal": achieved / 8000.0}
    if clocks and clocks.get("sm_mhz"):
        # clock-independent figures, so that rounds measured on boxes with different sustained clocks can be compared
        roofline["cycles_per_launch"] = avg_launch_s * clocks["sm_mhz"] * 1e6
        roofline["updates_per_clock"] = value / world * 1e9 / (clocks["sm_mhz"] * 1e6)
        roofline["clock_source"] = "median SM clock sampled by nvidia-smi during the timed region"

    # the second ceiling: the attempt arithmetic alone, no memory traffic, measured now on this device
    # in a 1 s run (so at the clock a long run holds); per GPU, like `achieved`
    from paper_2106_11286_b200 import probe_alu, probe_pipe
    from paper_2106_11286_b200.binding import PIPE_KINDS
    alu_peak = probe_alu(1.0, device) / 1e9
    pipe_rates = {name: round(probe_pipe(k, device), 3) for k, name in enumerate(PIPE_KINDS)}
    roofline["alu"] = {"bound": "alu", "achieved": value / world, "peak": alu_peak, "unit": UNIT, "frac": value / world / alu_peak,
                       "peak_source": "hb_probe_alu: Philox + proposal + neighbour sum on registers + delta-H + acceptance, "
                                      "4 attempts per thread as two packed pairs, 256-thread blocks, 4 per SM, measured in this run",
                       "pipe_rates": pipe_rates, "pipe_rates_unit": "warp-instructions per clock per SM (hb_probe_pipe, this run)"}

    # NEXT-1 beside the default: the same workload through the one-launch-per-colour kernel and through the fused
    # launches (all colour passes of 8 sweeps per launch), interleaved short runs after the timed region, and the rate of the
    # colour kernel with its HBM traffic folded into L2 (hb_probe_sc_l2: the ceiling of any scheme that only removes traffic)
    kernels = None
    if cfg["kind"] == "sc" and ctx.get_option("sc_kernel") >= 1 and "sc_kernel" not in options:
        def rate(kernel, sweeps=40):
            ctx.set_option("sc_kernel", kernel)
            ctx.sweep(T, 8)
            a, b = ev(), ev()
            a.record(); ctx.sweep(T, sweeps); b.record(); torch.cuda.synchronize()
            return float(n) * sweeps / (a.elapsed_time(b) * 1e-3) / 1e9
        try:
            default_kernel = ctx.get_option("sc_kernel")
            pairs = [(rate(1), rate(2)) for _ in range(3)]
            ctx.set_option("sc_kernel", default_kernel)
            kernels = {"unit": UNIT, "one_launch_per_colour (sc_kernel=1)": max(p[0] for p in pairs),
                       "fused_launches (sc_kernel=2, 8 sweeps per launch)": max(p[1] for p in pairs),
                       "note": "3 interleaved runs of 40 sweeps each, best of each; profiles/r02_c4_fused_full.md has the ncu comparison"}
            # the fold leaves the state undefined (re-initialised after each): interleaved with the default kernel, best of each
            fold = []
            for _ in range(3):
                fold.append((rate(default_kernel), ctx.probe_sc_l2(T, 40, 16) / 1e9))
                ctx.init_random()
                ctx.sweep(T, 8)
            kernels["hbm_traffic_folded_into_l2 (hb_probe_sc_l2)"] = max(f[1] for f in fold)
            kernels["default kernel beside the fold"] = max(f[0] for f in fold)
            kernels["fold_note"] = ("short runs (40 sweeps) after the probes, near boost clock: there the HBM traffic costs nothing and the fold's "
                                    "per-step address arithmetic shows; sustained at the power cap the fold gains 5-14 % (DESIGN.md section 7)")
        except Exception as exc:          # the fused launches need a row length the kernel takes
            kernels = {"unavailable": str(exc)}

    secondary = None
    if args.workload == "c4" and world == 1 and not args.no_workloads and not options:
        ctx.close()                       # the headline context is done: its memory goes back before the others are built
        try:
            secondary = run_secondary_workloads(device, local, peak, alu_peak)
        except Exception as exc:          # never lose the headline line to a secondary workload
            secondary = {"unavailable": repr(exc)}

    cpu = None if args.no_cpu_baseline else run_cpu_baseline(cfg)
    # acceptance rate of the timed sweeps themselves (reported with every timed config): hb_stats counts the
    # accepted moves inside the measuring passes, i.e. in the last sweep of every timed step
    acceptance = (stats1[1] - stats0[1]) / max(1, stats1[0] - stats0[0])

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": args.workload,
                   "lattice": "%s %s" % (cfg["kind"], cfg.get("L", cfg.get("R"))), "n_spins": n, "colours": n_colours,
                   "J": cfg["J"], "K": cfg["K"], "T": T, "start": cfg["start"], "seed": cfg["seed"],
                   "sweeps_per_step": SWEEPS_PER_STEP, "measurements_per_step": 1, "options": options,
                   "acceptance_rate": acceptance, "acceptance_counted_attempts": stats1[0] - stats0[0],
                   "l2": "state %.0f MB >> 126 MB L2: no flush between iterations" % (12.0 * n / 1e6)
                   if 12.0 * n > 4 * 126e6 else "state fits in L2: HBM roofline not meaningful",
                   "multi_gpu": "replicas only (seed + rank)"},
        "ns_per_update": 1.0 / value, "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
        "roofline": roofline, "cpu_baseline": cpu,
    }
    line["repeats"] = {"unit": UNIT, "values": repeat_values, "min": min(repeat_values), "median": statistics.median(repeat_values),
                       "max": max(repeat_values), "what": "%d timed regions of %d steps each, back to back; `value` is the first" % (len(repeat_values), args.steps)}
    if series_rate is not None:
        line["with_per_sweep_measurement"] = series_rate
    if kernels is not None:
        line["sc_kernels"] = kernels
    if secondary is not None:
        line["workloads"] = secondary
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
