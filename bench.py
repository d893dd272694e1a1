"""bench.py — throughput of the celstep hot path (one cel_transport = one pass of every SURVEY.md 8(a) row) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload config2] ...

A "step" is one whole transport of the workload's batch of events (init scan, reindex, action kernels, scoring,
push, non-blocking host loop, until no track and no initializer is left). The default workload is BASELINE.json
configs[1]: the 50-layer Pb/LAr sampling calorimeter, 1000 x 10 GeV e-, 2^20 track slots, sort mode by-action.
Prints ONE JSON line (rank 0). See DESIGN.md "Measurement" for every definition used here.

After the headline (outside its timed region) the default run also measures, on the same GPU: the other sort modes,
configs 1, 3, 4 at full size ("configs"), the config-5 slot-count x sort-mode sweep ("sweep"), and the oracle on the
host cores ("cpu_baseline", "cpu_baseline_legs").

N > 1 (torchrun, one rank per GPU): events are independent, so each rank transports its own batch of
the same size with its own seed and no data-path collective: weak scaling; value = all ranks' track-steps / max time;
the one exchange SURVEY.md 8(e) defines — the all_gather of the per-event tallies — is inside the e2e region.

--impl reference times the CPU oracle (oracle/, test infrastructure) as it stands on the host cores, on a bounded
sample of the same workload; it is a deliberately plain program, so the GPU/CPU ratio is context, not the headline.
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

from paper_2503_17608_b200 import workloads as W  # noqa: E402  (input data only)

SORT_NAMES = {0: "none", 1: "by_action", 2: "by_particle", 3: "partition", 4: "by_action_reuse"}
ACTIONS = ("PE", "PAIR", "COMPTON", "MOVE_G", "MOVE_C", "BREMS", "ANNIH", "VACANT")
STATE_BYTES = 64          # one slot's state: RecA + RecB
INDEX_BYTES = 4
HBM_NOMINAL_GBS = 8000.0  # the peak BASELINE.json's north_star names ("~8 TB/s")
MAX_SUBSTEPS = 0          # --max-substeps: 0 = the workload's own (10)
ACTION_KERNELS = ("annihilation", "photoelectric", "pair", "photon", "charged", "discrete")


def make_workload(name, n_events, n_slots, sort_mode, seed_offset=0):
    if name == "config1":
        w = W.config1(n_events=n_events or 1000, n_slots=n_slots or 4096, sort_mode=sort_mode, seed=1 + seed_offset)
    elif name == "config2":
        w = W.config2(n_events=n_events or 1000, n_slots=n_slots or (1 << 20), sort_mode=sort_mode, seed=2 + seed_offset)
    elif name == "config3":
        w = W.config3(n_events=n_events or 1000, n_slots=n_slots or (1 << 20), sort_mode=sort_mode, seed=3 + seed_offset)
    elif name == "config4":
        w = W.config4(n_events=n_events or 100, n_slots=n_slots or (1 << 22), sort_mode=sort_mode, seed=4 + seed_offset)
    elif name == "config5":
        w = W.config5(n_events=n_events or 2000, n_slots=n_slots or (1 << 20), sort_mode=sort_mode, seed=5 + seed_offset)
    else:
        raise SystemExit(f"unknown workload {name}")
    if MAX_SUBSTEPS:
        w.physics["max_substeps"] = MAX_SUBSTEPS       # PAPER.md:57 (fig. 1): the cap on chord substeps per iteration
        w.notes += f", max_substeps {MAX_SUBSTEPS}"
    return w


def describe(w):
    return (f"{w.name}: {w.n_events} events, {len(w.primaries)} primaries ({w.notes}), {w.n_slots} slots, "
            f"sort {SORT_NAMES[w.sort_mode]}, seed {w.physics['seed']}")


# ---------------------------------------------------------------- clocks during the timed region
class ClockSampler:
    """nvidia-smi sampling of SM clock and throttle reasons while the timed region runs (B200_PROFILING.md)."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu_index = gpu_index
        self.proc = None
        self.lines = []
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.gpu_index}", f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        def pump():
            for line in self.proc.stdout:
                self.lines.append(line.strip())
        self.thread = threading.Thread(target=pump, daemon=True)
        self.thread.start()

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()          # the exact process this object started
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(power)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------- the CPU oracle legs (cpu_baseline, --impl reference)
ORACLE_SAMPLES = {  # bounded samples of each workload for the plain CPU oracle: (events, slots)
    "config1": (1000, 4096), "config2": (200, 1 << 18), "config3": (200, 1 << 18), "config4": (1, 1 << 17), "config5": (200, 1 << 18),
}


def oracle_sample_workload(workload, sort_mode, events=0, slots=0, oracle_events=0, oracle_slots=0):
    """a bounded sample of a workload for the oracle: fewer events of the same kind in fewer slots (the oracle visits
    every slot in every phase of every iteration; its result is slot-count independent up to the history keying)"""
    full = make_workload(workload, events, slots, sort_mode)
    d_ev, d_sl = ORACLE_SAMPLES[workload]
    n_ev = max(1, min(full.n_events, oracle_events or d_ev))
    n_sl = oracle_slots or min(d_sl, full.n_slots)
    per_event = len(full.primaries) // full.n_events
    w = make_workload(workload, n_ev, n_sl, sort_mode)
    w.primaries = full.primaries[: n_ev * per_event].copy()
    sample = (f"{n_ev} of {full.n_events} events of {full.name} ({per_event} primaries/event), {n_sl} slots, "
              f"sort {SORT_NAMES[w.sort_mode]}, g++ -O2 -ffp-contract=off -fopenmp")
    return w, sample


def time_oracle(w, threads=1):
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import oracle as orc   # test infrastructure; this leg is one of the three places allowed to run it
    o = orc.Oracle(w.geometry, w.materials, w.physics, w.n_slots, w.sort_mode)
    o.set_threads(threads)
    t0 = time.perf_counter()
    o.transport(w.primaries, w.n_events)
    dt = time.perf_counter() - t0
    c = o.counters()
    o.close()
    return dt, int(c["track_steps"])


def oracle_legs(args, workloads):
    """the oracle as it stands on the host cores: one thread and all cores (OpenMP over slots in the per-slot phases,
    bit-identical results), on a bounded sample of each workload"""
    nproc = os.cpu_count() or 1
    legs = []
    for name in workloads:
        extra = (args.events, args.slots, args.oracle_events, args.oracle_slots) if name == args.workload else ()
        ow, sample = oracle_sample_workload(name, 1, *extra)
        for threads in sorted({1, nproc}):
            dt, ts = time_oracle(ow, threads)
            legs.append({"workload": name, "value": ts / dt, "unit": "track-steps/s", "cores": threads, "nproc": nproc, "kind": "oracle",
                         "sample": sample, "seconds": round(dt, 2), "events_per_s": ow.n_events / dt})
    return legs


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w, sample = oracle_sample_workload(args.workload, args.sort_mode, args.events, args.slots, args.oracle_events, args.oracle_slots)
    threads = args.oracle_threads or (os.cpu_count() or 1)
    for _ in range(args.warmup):
        time_oracle(w, threads)
    total_t, total_steps = 0.0, 0
    for _ in range(args.steps):
        dt, ts = time_oracle(w, threads)
        total_t += dt; total_steps += ts
    value = total_steps / total_t
    full = make_workload(args.workload, args.events, args.slots, args.sort_mode)
    out = {
        "impl": "reference", "metric": "track-steps/s", "value": value, "unit": "track-steps/s",
        "events_per_s": w.n_events * args.steps / total_t,
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total_t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": describe(full), "sample_per_step": sample},
        "cpu_baseline": {"value": value, "unit": "track-steps/s", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "track-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out))
    return 0


# ---------------------------------------------------------------- algorithmic bytes per kernel
def algorithmic_bytes(counts, n_slots, sort_mode, n_initialised, n_secondaries):
    """bytes each kernel MUST move over one whole transport, from the per-iteration action counts the library logs
    (64 B state, 4 B index, 1 B key, 64 B per staged secondary; tally atomics stay in L2).
    counts: [iterations][8] action counts after P1. Returns {kernel name: bytes}."""
    c = counts.astype(np.float64).sum(0)
    it = float(len(counts))
    idx = INDEX_BYTES if sort_mode in (1, 2, 4) else 0
    rw = 2 * STATE_BYTES + idx          # gather + write back one slot through the index
    n = float(n_slots)
    sec = float(n_secondaries)
    out = {
        # key bytes read once (an UPPER bound: tiles that are entirely vacant and get no fill are skipped) + (read init,
        # write slot) per initialised track + one index per non-vacant slot
        "fill_sort": it * n * 1 + float(n_initialised) * 2 * STATE_BYTES + (it * n - c[7]) * idx,
        "annihilation": c[6] * (rw + 2 * STATE_BYTES),
        "photoelectric": c[0] * (rw + STATE_BYTES),
        "pair": c[1] * (rw + 2 * STATE_BYTES),
        "photon": (c[3] + c[2]) * rw + c[2] * STATE_BYTES,                   # Compton stages one electron
        "charged": (c[4] + c[5]) * rw + c[5] * STATE_BYTES,                  # bremsstrahlung stages one photon
        "push": sec * (1 + 2 * STATE_BYTES),                                 # nsec byte + (read staging, write stack)
    }
    # sort mode 3: two passes over the popped initializers (8 B meta each), 4 B pop position written, then read by the fill
    out["part_count"] = float(n_initialised) * 8
    out["part_scatter"] = float(n_initialised) * (8 + INDEX_BYTES)
    if sort_mode == 3:
        out["fill_sort"] += float(n_initialised) * INDEX_BYTES
    out["discrete"] = sum(out[k] for k in ("annihilation", "photoelectric", "pair"))
    out["hits_flush"] = 0.0
    return out


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_profile_table(fname):
    """rows of a committed ncu summary table under profiles/ (`#` comments; whitespace-separated columns, first = kernel)"""
    path = os.path.join(ROOT, "profiles", fname)
    rows = {}
    if os.path.exists(path):
        with open(path) as f:
            for line in f:
                parts = line.split()
                if parts and not line.startswith("#"):
                    rows[parts[0]] = parts[1:]
    return rows


# ---------------------------------------------------------------- the CUDA arm
def run_cuda(args):
    import torch
    import torch.distributed as dist
    from paper_2503_17608_b200 import binding, sharding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    binding.load_library()   # raises if libcelstep.so has not been built

    stream = torch.cuda.Stream(device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)       # > 126 MB L2
    peak, peak_kind = measured_peaks()

    def make_ctx(w, sort_mode):
        cap = w.physics["init_capacity"] or max(8 * w.n_slots, 1 << 24)
        nbytes = binding.workspace_bytes(w.n_slots, cap, sort_mode)
        buf = torch.empty(nbytes + 256, dtype=torch.uint8, device=dev)   # torch owns the device memory
        ptr = (buf.data_ptr() + 255) // 256 * 256
        ctx = binding.from_workload(w, sort_mode=sort_mode, stream=stream.cuda_stream, workspace=ptr, workspace_bytes=nbytes)
        ctx._buf = buf
        return ctx

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed_steps(ctx, w, d_prim, n, resident=True):
        """n steps, each bracketed by CUDA events on the launch stream; L2 flushed between steps (outside the events)"""
        ms, steps, launches, v = 0.0, 0, 0, None
        with torch.cuda.stream(stream):
            for _ in range(n):
                flush.fill_(1)
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                if resident:
                    ctx.transport_device(d_prim.data_ptr(), len(w.primaries), w.n_events)
                else:
                    ctx.transport(w.primaries, w.n_events)
                e1.record(stream)
                v = ctx.tallies_view()      # synchronises the stream
                ms += e0.elapsed_time(e1)
                steps += v["track_steps"]; launches += v["kernel_launches"]
        return ms, steps, launches, v

    def profile_pass(ctx, w, d_prim):
        """per-kernel device time: one more transport of the same workload in the library's profile mode (direct launches
        with a CUDA event after every kernel on the launch stream) -> {kernel: ms, launches, share, alg_bytes, gbs, frac}"""
        ctx.set_option("profile", 1)
        with torch.cuda.stream(stream):
            flush.fill_(1)
            ctx.transport_device(d_prim.data_ptr(), len(w.primaries), w.n_events)
            pview = ctx.tallies_view()
        ktimes = ctx.kernel_times()
        counts = ctx.counts()
        ctx.set_option("profile", 0)
        alg = algorithmic_bytes(counts, w.n_slots, ctx.sort_mode, len(w.primaries) + pview["secondaries"], pview["secondaries"])
        total_ms = sum(t for t, _ in ktimes.values()) or 1.0
        kernels = {}
        for name, (kms, kl) in ktimes.items():
            if kl == 0:
                continue
            gbs = alg[name] / (kms * 1e-3) / 1e9 if kms > 0 else 0.0
            kernels[name] = {"ms": round(kms, 4), "launches": kl, "share": round(kms / total_ms, 4), "alg_bytes": alg[name],
                             "gbs": round(gbs, 2), "frac": round(gbs / peak, 4), "frac_nominal": round(gbs / HBM_NOMINAL_GBS, 4)}
        return kernels, counts, pview

    def measure(w, sort_mode, steps, warmup, with_profile=True):
        """one workload in one sort mode: throughput + (optionally) the dominant kernel's HBM fraction"""
        ctx = make_ctx(w, sort_mode)
        d_prim = torch.from_numpy(w.primaries.view(np.uint8).copy()).to(dev)
        timed_steps(ctx, w, d_prim, warmup)
        ms, ts, _, v = timed_steps(ctx, w, d_prim, steps)
        out = {"track_steps_per_s": ts / (ms * 1e-3), "events_per_s": w.n_events * steps / (ms * 1e-3), "ms_per_step": ms / steps,
               "iterations": int(v["iterations"]), "track_steps_per_step": ts / steps}
        if with_profile:
            kernels, _, _ = profile_pass(ctx, w, d_prim)
            dom = max(kernels, key=lambda k: kernels[k]["ms"])
            out["dominant_kernel"] = dom
            out["dominant_hbm_frac"] = kernels[dom]["frac"]
            out["hbm_frac"] = {k: kernels[k]["frac"] for k in kernels}
        ctx.close()
        del d_prim
        return out

    # ================================================================ the headline: args.workload (config 2), timed
    w = make_workload(args.workload, args.events, args.slots, args.sort_mode, seed_offset=1000 * rank)
    d_prim = torch.from_numpy(w.primaries.view(np.uint8).copy()).to(dev)  # inputs resident in HBM for `value`
    ctx = make_ctx(w, w.sort_mode)
    timed_steps(ctx, w, d_prim, args.warmup)
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    ms, track_steps, launches, view = timed_steps(ctx, w, d_prim, args.steps)
    barrier()
    clocks = sampler.stop() if rank == 0 else None

    # e2e: the same steps through the public call with HOST primaries, H2D copy and tally D2H inside the timed region;
    # with several ranks also the one exchange SURVEY.md 8(e) defines: the all_gather of the per-event tallies
    barrier()
    t0 = time.perf_counter()
    e2e_steps = 0
    merged = None
    with torch.cuda.stream(stream):
        for _ in range(args.steps):
            ctx.transport(w.primaries, w.n_events)
            v = ctx.tallies_view()
            e2e_steps += v["track_steps"]
            if world > 1:
                merged = sharding.merge_tallies(v["fixed"], world * w.n_events, device=dev)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    h2d = int(w.primaries.nbytes)
    d2h = int(v["fixed"].nbytes)
    if merged is not None:   # every rank's events are there, each conserving its primary energy (S10)
        e = merged.astype(np.float64).sum(1) * 2.0 ** -36
        assert merged.shape[0] == world * w.n_events and np.all(np.abs(e - e[0]) <= 1e-9 * e[0]), "merged tallies"

    if world > 1:
        ms, e2e_s = sharding.max_over_ranks(ms, device=dev), sharding.max_over_ranks(e2e_s, device=dev)
        track_steps = sharding.sum_over_ranks(track_steps, device=dev)
        e2e_steps = sharding.sum_over_ranks(e2e_steps, device=dev)
        launches = sharding.sum_over_ranks(launches, device=dev)
    if rank != 0:
        ctx.close()
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- per-kernel device time and the rooflines of the dominant kernel
    kernels, counts, pview = profile_pass(ctx, w, d_prim)
    dominant = max(kernels, key=lambda k: kernels[k]["ms"])
    dk = kernels[dominant]
    # the committed ncu captures are of the default workload (config 2, by action, 2^20 slots): no ncu figure for others
    is_default = args.workload == "config2" and w.sort_mode == 1 and not args.events and not args.slots and not args.max_substeps
    traffic = traffic_it = alg_at_it = None
    traffic_source = None
    if is_default:
        row = load_profile_table("traffic_r02.txt").get(dominant)
        if row:
            traffic, traffic_it = float(row[0]), int(row[1])
            traffic_source = "profiles/traffic_r02.txt (builder's ncu --set full capture of that iteration; not measured in this run)"
            if traffic_it < len(counts) and dominant in ACTION_KERNELS:
                alg_at_it = algorithmic_bytes(counts[traffic_it:traffic_it + 1], w.n_slots, w.sort_mode, 0, 0)[dominant]
    roofline = {"bound": "hbm", "bound_measured": "fp64 dependent chains / latency (see roofline_alu; DESIGN.md section 7)",
                "kernel": dominant, "achieved": dk["gbs"], "peak": peak, "unit": "GB/s",
                "frac": dk["frac"], "frac_nominal_8TBs": dk["frac_nominal"], "traffic": traffic, "traffic_iteration": traffic_it,
                "traffic_source": traffic_source,
                "alg_bytes_at_traffic_iteration": alg_at_it, "peak_kind": peak_kind,
                "alg_bytes_per_launch": dk["alg_bytes"] / dk["launches"], "avg_launch_us": 1e3 * dk["ms"] / dk["launches"],
                "share_of_step": dk["share"], "iterations": int(pview["iterations"]),
                "how": "profile pass after the timed steps: same workload, CUDA events around every kernel launch"}
    # the bound that binds (SURVEY.md 8(d) "secondary bound to report"): issue slots. Thread instructions per track and the
    # pipe utilisations come from the committed ncu capture; the track rate and the clock are this run's.
    roofline_alu = None
    if is_default:
        row = load_profile_table("alu_r02.txt").get(dominant)
        tracks = {"charged": counts[:, 4].sum() + counts[:, 5].sum(), "photon": counts[:, 2].sum() + counts[:, 3].sum()}.get(dominant)
        if row and tracks:
            warp_inst, thr_per_inst, n_tracks, issue_busy, fp64_active = (float(x) for x in row[:5])
            sm_mhz = (clocks or {}).get("sm_mhz") or 1965.0
            inst_per_track = warp_inst * thr_per_inst / n_tracks
            achieved = inst_per_track * float(tracks) / (dk["ms"] * 1e-3)
            alu_peak = 148 * 4 * 32 * sm_mhz * 1e6      # SMs x schedulers x lanes x clock: thread instructions / s
            roofline_alu = {"bound": "alu", "kernel": dominant, "warp_inst_per_track": warp_inst / n_tracks,
                            "thread_inst_per_track": inst_per_track, "issue_slots_busy": issue_busy / 100.0,
                            "fp64_pipe_active": fp64_active / 100.0, "achieved_thread_inst_per_s": achieved, "peak": alu_peak,
                            "unit": "thread instructions/s", "frac": achieved / alu_peak, "sm_mhz": sm_mhz,
                            "source": "profiles/alu_r02.txt (builder's ncu --set full capture, command in profiles/iter101_r02.md) "
                                      "x this run's track rate and SM clock; peak = 148 SMs x 4 schedulers x 32 lanes x clock"}

    # ---- the other sort modes (BASELINE.json metric: per sort mode)
    per_mode = {}
    if not args.no_modes:
        for mode in (0, 1, 2, 3, 4):
            if mode == w.sort_mode:
                per_mode[SORT_NAMES[mode]] = {"track_steps_per_s": track_steps / (ms * 1e-3) / world, "events_per_s": w.n_events * args.steps / (ms * 1e-3)}
                continue
            m = measure(w, mode, max(1, min(args.steps, 3)), 1, with_profile=False)
            per_mode[SORT_NAMES[mode]] = {"track_steps_per_s": m["track_steps_per_s"], "events_per_s": m["events_per_s"]}
    ctx.close()

    # ---- configs 1, 3, 4 at full size and the config-5 sweep (BASELINE.json configs[0..4]); world == 1 only
    configs, sweep = None, None
    if world == 1 and not args.no_configs:
        configs = {}
        for name in ("config1", "config3", "config4"):
            if name == args.workload:
                continue
            wc = make_workload(name, 0, 0, 1)
            configs[name] = dict(measure(wc, 1, 3, 1), workload=describe(wc))
    if world == 1 and not args.no_sweep:
        sweep = []
        for log2n in (16, 18, 20, 22, 24):
            for mode in (0, 1, 2):
                w5 = make_workload("config5", 0, 1 << log2n, mode)
                m = measure(w5, mode, 2, 1)
                sweep.append({"slots_log2": log2n, "sort": SORT_NAMES[mode], "track_steps_per_s": m["track_steps_per_s"],
                              "events_per_s": m["events_per_s"], "iterations": m["iterations"], "ms_per_step": m["ms_per_step"],
                              "dominant_kernel": m["dominant_kernel"], "dominant_hbm_frac": m["dominant_hbm_frac"],
                              "hbm_frac": m["hbm_frac"]})

    cpu_baseline, cpu_legs = None, None
    if world == 1 and not args.no_cpu_baseline:
        names = [args.workload] + ([n for n in ("config1", "config3", "config4") if n != args.workload] if not args.no_configs else [])
        cpu_legs = oracle_legs(args, names)
        head = [l for l in cpu_legs if l["workload"] == args.workload]
        best = max(head, key=lambda l: l["value"])
        cpu_baseline = {k: best[k] for k in ("value", "unit", "cores", "nproc", "kind", "sample", "seconds", "events_per_s")}

    value = track_steps / (ms * 1e-3)
    out = {
        "metric": "track-steps/s", "value": value, "unit": "track-steps/s",
        "events_per_s": world * w.n_events * args.steps / (ms * 1e-3),
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": describe(w), "per_rank": world > 1, "l2": "flushed between steps (256 MB write)",
                   "track_steps_per_step": track_steps / args.steps / world, "iterations_per_step": int(view["iterations"]),
                   "timing": "CUDA events on the launch stream around each cel_transport_device; primaries resident in HBM"},
        "e2e": {"value": e2e_steps / e2e_s, "unit": "track-steps/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": 1e3 * e2e_s / args.steps,
                "how": "cel_transport(host primaries) + cel_tallies (tally D2H) per step" +
                       (" + all_gather of the per-event tallies over the ranks (NCCL)" if world > 1 else "") + ", host wall clock"},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": roofline,
        "roofline_alu": roofline_alu,
        "kernels": kernels,
        "per_sort_mode": per_mode,
        "configs": configs,
        "sweep": sweep,
        "cpu_baseline": cpu_baseline,
        "cpu_baseline_legs": cpu_legs,
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="config2", choices=["config1", "config2", "config3", "config4", "config5"])
    ap.add_argument("--events", type=int, default=0, help="override the workload's number of events")
    ap.add_argument("--slots", type=int, default=0, help="override the workload's number of track slots")
    ap.add_argument("--sort-mode", type=int, default=1, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--no-modes", action="store_true", help="skip the other sort modes")
    ap.add_argument("--no-configs", action="store_true", help="skip configs 1, 3, 4")
    ap.add_argument("--no-sweep", action="store_true", help="skip the config-5 slot-count x sort-mode sweep")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--quick", action="store_true", help="= --no-modes --no-configs --no-sweep --no-cpu-baseline")
    ap.add_argument("--oracle-events", type=int, default=0, help="events in the oracle's bounded sample (0 = the workload's default sample)")
    ap.add_argument("--oracle-slots", type=int, default=0)
    ap.add_argument("--oracle-threads", type=int, default=0, help="--impl reference: host threads (0 = all cores)")
    ap.add_argument("--max-substeps", type=int, default=0, help="override the cap on helix chord substeps per iteration (PAPER.md:57)")
    args = ap.parse_args()
    if args.quick:
        args.no_modes = args.no_configs = args.no_sweep = args.no_cpu_baseline = True
    global MAX_SUBSTEPS
    MAX_SUBSTEPS = args.max_substeps
    if args.warmup < 3 and args.impl == "cuda":
        print("bench.py: warning: fewer than 3 warm-up steps", file=sys.stderr)
    return run_reference(args) if args.impl == "reference" else run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
