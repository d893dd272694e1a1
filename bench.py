"""bench.py — throughput of the celstep hot path (one cel_transport = one pass of every SURVEY.md 8(a) row) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload config2] ...

A "step" is one whole transport of the workload's batch of events (init scan, reindex, action kernels, scoring,
push, non-blocking host loop, until no track and no initializer is left). The default workload is BASELINE.json
configs[1]: the 50-layer Pb/LAr sampling calorimeter, 1000 x 10 GeV e-, 2^20 track slots, sort mode by-action.
Prints ONE JSON line (rank 0). See DESIGN.md "Measurement" for every definition used here.

N > 1 (torchrun, one rank per GPU): events are independent, so each rank transports its own batch of
the same size with its own seed and no data-path collective: weak scaling; value = all ranks' track-steps / max time.

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
MAX_SUBSTEPS = 0        # --max-substeps: 0 = the workload's own (10)


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
def oracle_sample_workload(args):
    """a bounded sample of the benchmark workload for the single-threaded oracle: fewer events of the same kind in
    fewer slots (the oracle visits every slot in every phase of every iteration; its result is slot-count independent
    up to the history keying)"""
    full = make_workload(args.workload, args.events, args.slots, args.sort_mode)
    n_ev = max(1, min(full.n_events, args.oracle_events))
    per_event = len(full.primaries) // full.n_events
    w = make_workload(args.workload, n_ev, args.oracle_slots, args.sort_mode)
    w.primaries = full.primaries[: n_ev * per_event].copy()
    sample = (f"{n_ev} of {full.n_events} events of {full.name} ({per_event} primaries/event), "
              f"{args.oracle_slots} slots, sort {SORT_NAMES[w.sort_mode]}, 1 thread, g++ -O2 -ffp-contract=off")
    return w, sample


def time_oracle(w):
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import oracle as orc   # test infrastructure; this leg is one of the three places allowed to run it
    o = orc.Oracle(w.geometry, w.materials, w.physics, w.n_slots, w.sort_mode)
    t0 = time.perf_counter()
    o.transport(w.primaries, w.n_events)
    dt = time.perf_counter() - t0
    c = o.counters()
    o.close() if hasattr(o, "close") else None
    return dt, int(c["track_steps"])


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w, sample = oracle_sample_workload(args)
    for _ in range(args.warmup):
        time_oracle(w)
    total_t, total_steps = 0.0, 0
    for _ in range(args.steps):
        dt, ts = time_oracle(w)
        total_t += dt; total_steps += ts
    value = total_steps / total_t
    full = make_workload(args.workload, args.events, args.slots, args.sort_mode)
    out = {
        "impl": "reference", "metric": "track-steps/s", "value": value, "unit": "track-steps/s",
        "events_per_s": w.n_events * args.steps / total_t,
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total_t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": describe(full), "sample_per_step": sample},
        "cpu_baseline": {"value": value, "unit": "track-steps/s", "cores": 1, "kind": "oracle", "sample": sample},
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
        # key bytes read once (an upper bound: tiles that are entirely vacant and get no fill are skipped) + (read init,
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
    return out


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_profile_traffic(kernel):
    """(dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel`, iteration captured) from the committed
    ncu --set full summary (profiles/traffic.txt: lines `kernel_name bytes_per_launch iteration`), or (None, None)"""
    path = os.path.join(ROOT, "profiles", "traffic.txt")
    if not os.path.exists(path):
        return None, None
    with open(path) as f:
        for line in f:
            parts = line.split()
            if len(parts) >= 2 and not line.startswith("#") and parts[0] == kernel:
                return float(parts[1]), (int(parts[2]) if len(parts) > 2 else None)
    return None, None


# ---------------------------------------------------------------- the CUDA arm
def run_cuda(args):
    import torch
    import torch.distributed as dist
    from paper_2503_17608_b200 import binding

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

    w = make_workload(args.workload, args.events, args.slots, args.sort_mode, seed_offset=1000 * rank)
    stream = torch.cuda.Stream(device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)       # > 126 MB L2
    d_prim = torch.from_numpy(w.primaries.view(np.uint8).copy()).to(dev)  # inputs resident in HBM for `value`
    h_prim = w.primaries                                                  # host buffer for `e2e`

    def make_ctx(sort_mode):
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

    def timed_steps(ctx, n, resident=True):
        """n steps, each bracketed by CUDA events on the launch stream; L2 flushed between steps (outside the events)"""
        ms, steps, launches = 0.0, 0, 0
        with torch.cuda.stream(stream):
            for _ in range(n):
                flush.fill_(1)
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                if resident:
                    ctx.transport_device(d_prim.data_ptr(), len(w.primaries), w.n_events)
                else:
                    ctx.transport(h_prim, w.n_events)
                e1.record(stream)
                v = ctx.tallies_view()      # synchronises the stream
                ms += e0.elapsed_time(e1)
                steps += v["track_steps"]; launches += v["kernel_launches"]
        return ms, steps, launches, v

    ctx = make_ctx(w.sort_mode)
    timed_steps(ctx, args.warmup)
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    ms, track_steps, launches, view = timed_steps(ctx, args.steps)
    barrier()
    clocks = sampler.stop() if rank == 0 else None

    # e2e: the same steps through the public call with HOST primaries, H2D copy and tally D2H inside the timed region
    barrier()
    t0 = time.perf_counter()
    e2e_steps = 0
    with torch.cuda.stream(stream):
        for _ in range(args.steps):
            ctx.transport(h_prim, w.n_events)
            v = ctx.tallies_view()
            e2e_steps += v["track_steps"]
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    h2d = int(h_prim.nbytes)
    d2h = int(v["fixed"].nbytes)

    if world > 1:
        t = torch.tensor([ms, e2e_s], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms, e2e_s = float(t[0]), float(t[1])
        s = torch.tensor([track_steps, e2e_steps, launches], dtype=torch.float64, device=dev)
        dist.all_reduce(s, op=dist.ReduceOp.SUM)
        track_steps, e2e_steps, launches = float(s[0]), float(s[1]), float(s[2])
    if rank != 0:
        ctx.close()
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- per-kernel device time: one more transport of the same workload in the library's profile mode (direct
    # launches with a CUDA event after every kernel on the launch stream); the dominant kernel gives `roofline`
    ctx.set_option("profile", 1)
    with torch.cuda.stream(stream):
        flush.fill_(1)
        ctx.transport_device(d_prim.data_ptr(), len(w.primaries), w.n_events)
        pview = ctx.tallies_view()
    ktimes = ctx.kernel_times()
    counts = ctx.counts()
    ctx.set_option("profile", 0)
    alg = algorithmic_bytes(counts, w.n_slots, w.sort_mode, len(w.primaries) + pview["secondaries"], pview["secondaries"])
    peak, peak_kind = measured_peaks()
    total_kernel_ms = sum(t for t, _ in ktimes.values()) or 1.0
    kernels = {}
    for name, (kms, kl) in ktimes.items():
        if kl == 0:
            continue
        gbs = alg[name] / (kms * 1e-3) / 1e9 if kms > 0 else 0.0
        kernels[name] = {"ms": round(kms, 4), "launches": kl, "share": round(kms / total_kernel_ms, 4),
                         "alg_bytes": alg[name], "gbs": round(gbs, 2), "frac": round(gbs / peak, 4)}
    dominant = max(kernels, key=lambda k: kernels[k]["ms"])
    dk = kernels[dominant]
    # the committed ncu capture is of the default workload (config 2, by action, 2^20 slots): no traffic figure for others
    is_default = args.workload == "config2" and w.sort_mode == 1 and not args.events and not args.slots and not args.max_substeps
    traffic, traffic_it = load_profile_traffic(dominant) if is_default else (None, None)
    alg_at_it = None
    if traffic_it is not None and traffic_it < len(counts) and dominant in ("annihilation", "photoelectric", "pair", "photon", "charged", "discrete"):
        alg_at_it = algorithmic_bytes(counts[traffic_it:traffic_it + 1], w.n_slots, w.sort_mode, 0, 0)[dominant]
    roofline = {"bound": "hbm", "kernel": dominant, "achieved": dk["gbs"], "peak": peak, "unit": "GB/s",
                "frac": dk["frac"], "traffic": traffic, "traffic_iteration": traffic_it,
                "alg_bytes_at_traffic_iteration": alg_at_it, "peak_kind": peak_kind,
                "alg_bytes_per_launch": dk["alg_bytes"] / dk["launches"], "avg_launch_us": 1e3 * dk["ms"] / dk["launches"],
                "share_of_step": dk["share"], "iterations": int(pview["iterations"]),
                "how": "profile pass after the timed steps: same workload, CUDA events around every kernel launch"}

    # ---- the other sort modes (BASELINE.json metric: per sort mode)
    per_mode = {}
    if not args.no_modes:
        for mode in (0, 1, 2, 3, 4):
            if mode == w.sort_mode:
                per_mode[SORT_NAMES[mode]] = {"track_steps_per_s": track_steps / (ms * 1e-3) / world if world > 1 else track_steps / (ms * 1e-3),
                                              "events_per_s": w.n_events * args.steps / (ms * 1e-3)}
                continue
            c2 = make_ctx(mode)
            timed_steps(c2, 1)
            m_ms, m_steps, _, _ = timed_steps(c2, max(1, min(args.steps, 3)))
            per_mode[SORT_NAMES[mode]] = {"track_steps_per_s": m_steps / (m_ms * 1e-3),
                                          "events_per_s": w.n_events * max(1, min(args.steps, 3)) / (m_ms * 1e-3)}
            c2.close()
    ctx.close()

    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        ow, sample = oracle_sample_workload(args)
        dt, ts = time_oracle(ow)
        cpu_baseline = {"value": ts / dt, "unit": "track-steps/s", "cores": 1, "kind": "oracle", "sample": sample,
                        "seconds": round(dt, 2), "events_per_s": ow.n_events / dt}

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
                "how": "cel_transport(host primaries) + cel_tallies (tally D2H) per step, host wall clock"},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": roofline,
        "kernels": kernels,
        "per_sort_mode": per_mode,
        "cpu_baseline": cpu_baseline,
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
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--oracle-events", type=int, default=200, help="events in the oracle's bounded sample")
    ap.add_argument("--oracle-slots", type=int, default=1 << 18)
    ap.add_argument("--max-substeps", type=int, default=0, help="override the cap on helix chord substeps per iteration (PAPER.md:57)")
    args = ap.parse_args()
    global MAX_SUBSTEPS
    MAX_SUBSTEPS = args.max_substeps
    if args.warmup < 3 and args.impl == "cuda":
        print("bench.py: warning: fewer than 3 warm-up steps", file=sys.stderr)
    return run_reference(args) if args.impl == "reference" else run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
