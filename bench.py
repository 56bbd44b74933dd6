#!/usr/bin/env python
"""bench.py — throughput of the event-based transport hot path on B200.

A step = one pass of the whole hot path (source, flights with track-length tally,
collisions, census, comb, batch close-out) over one batch of the workload; default
workload = BASELINE.json config 5 (64^3 voxel box, 7 groups, 20 census steps + comb)
at its full batch size of 1e7 histories.  Prints ONE JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--n-hist 10000000]
    python bench.py --impl reference ...      # times the CPU oracle on a bounded sample
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import mcdc_inputs as mi  # noqa: E402

METRIC = "histories/sec"
UNIT = "histories/s"
FULL_N = {1: 100_000, 2: 1_000_000, 3: 1_000_000, 4: 1_000_000, 5: 10_000_000}
ORACLE_SAMPLE_N = {1: 4_000_000, 2: 2_000_000, 3: 600_000, 4: 4_000_000, 5: 200_000}


DOGLEG = 0   # --dogleg SUB: the dog-leg void duct stand-in with SUB tally bins per cell and axis
DN = None    # --delayed: (beta, time_scale) of the seeded six-group delayed-neutron set (DESIGN.md C.16)
IC = None    # --implicit-capture: (w_roulette, w_survive) (DESIGN.md C.15)
EIG = None   # --eigenvalue: (n_inactive, n_active) of the pin-cell k-eigenvalue workload (DESIGN.md C.14)


def make_cfg(k, n_hist, seed=0):
    if DOGLEG:
        cfg = mi.dogleg_duct(n_hist=n_hist, n_batch=1, seed=seed, sub=DOGLEG)
        return mi.implicit_capture(cfg, *IC) if IC else cfg
    if EIG:
        return mi.pin_cell_eigenvalue(n_hist=n_hist, n_inactive=EIG[0], n_active=EIG[1], n_batch=1, seed=seed)
    cfg = mi.config(k, n_hist=n_hist, n_batch=1, seed=seed)
    if DN:
        cfg = mi.seeded_delayed(cfg, beta=DN[0], time_scale=DN[1])
    return mi.implicit_capture(cfg, *IC) if IC else cfg


def workload_name(k, n_hist):
    if DOGLEG:
        return (f"dog-leg void duct stand-in (PAPER.md:79-83: v = 1 cm/s, source on for 50 s, flux to 200 s): 6x10x6 cells of "
                f"10 cm, {6 * DOGLEG}x{10 * DOGLEG}x{6 * DOGLEG}x20 tally, one batch of {n_hist} histories per step" +
                (f", implicit capture (roulette below {IC[0]} to {IC[1]})" if IC else ", analog"))
    if EIG:
        return (f"pin-cell k-eigenvalue (stand-in for PAPER.md:91): {EIG[0]} inactive + {EIG[1]} active cycles of "
                f"{n_hist} particles, 20x20x100x7 tally; a history = one particle of one cycle")
    return (f"config{k}: BASELINE.json configs[{k - 1}], one batch of {n_hist} histories per step" +
            (f" + implicit capture (roulette below {IC[0]} to {IC[1]}), weighted comb" if IC else "") +
            (f" + 6 delayed-neutron groups (beta {DN[0]}, decay constants 0.0125..3 / {DN[1]} s)" if DN else ""))


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region.  start() returns once the first
    sample has arrived; stop() waits for one more, so that even a timed region shorter than the sampling
    period (configs 1-3) carries samples taken while the GPU was under this load."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0, period_ms=100):
        self.lines, self.proc, self.t_mark = [], None, None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", str(period_ms),
                 "-i", str(index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
            t0 = time.perf_counter()
            while not self.lines and time.perf_counter() - t0 < 5.0:
                time.sleep(0.01)
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def mark(self):
        """Start of the timed region: only samples from here on are counted."""
        self.t_mark = time.perf_counter()

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"], "samples": 0}
        n0, t0 = len(self.lines), time.perf_counter()
        while len(self.lines) == n0 and time.perf_counter() - t0 < 1.0:
            time.sleep(0.01)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            pass
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ts, ln in self.lines:
            if self.t_mark is not None and ts < self.t_mark:
                continue
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(mx)) if mx else None, "reasons": sorted(reasons),
                "samples": len(sm)}


def measured_peak_hbm():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def issue_peak():
    """Warp-instruction issue peak: 148 SMs x 4 SM sub-partitions x 1 warp
    instruction per clock x the maximum SM clock."""
    mhz, src = 1965.0, "148 SMs x 4 SMSPs x 1 inst/clk x 1965 MHz"
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            mhz = float(json.load(f).get("sm_max_mhz", mhz))
        src = f"148 SMs x 4 SMSPs x 1 inst/clk x {mhz:.0f} MHz (MEASURED_PEAKS.json sm_max_mhz)"
    return 148 * 4 * mhz * 1e6 / 1e9, src


EVENT_MODEL = "128 B/flight + 88 B/collision + 80 B/secondary + 72 B/surface event + 160 B/census (SURVEY 8(d))"


def event_model_bytes(c):
    """HBM bytes the per-event-kernel form of the path moves: the state of a particle
    goes through HBM once per event."""
    return (128 * c["flights"] + 88 * c["collisions"] + 80 * c["secondaries"] +
            72 * (c["crossings"] + c["reflections"]) + 160 * c["census"])


def run_oracle_sample(k, n_hist, seed=0):
    """The oracle as it stands, single thread, on a bounded sample of the workload."""
    from oracle import Oracle
    cfg = make_cfg(k, n_hist, seed)
    o = Oracle(cfg)
    t0 = time.perf_counter()
    o.run()
    dt = time.perf_counter() - t0
    c = o.counters()
    o.close()
    return dt, c


def _oracle_worker(args):
    k, n, seed, glob = args
    global DOGLEG, DN, IC, EIG
    DOGLEG, DN, IC, EIG = glob
    dt, c = run_oracle_sample(k, n, seed)
    return dt, c["segments"], c["flights"]


def run_oracle_all_cores(k, n_hist):
    """one oracle process per batch (batches are independent streams) across the host's
    cores, each on the same bounded sample with its own seed; aggregate histories/s."""
    import multiprocessing as mp
    avail = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    procs = max(1, min(avail, 16))                      # (each config-5 process holds 1.3 GB of tally arrays)
    ctx = mp.get_context("spawn")
    t0 = time.perf_counter()
    with ctx.Pool(procs) as pool:
        res = pool.map(_oracle_worker, [(k, n_hist, 100 + i, (DOGLEG, DN, IC, EIG)) for i in range(procs)])
    wall = time.perf_counter() - t0
    gens = sum(EIG) if EIG else 1
    busy = max(r[0] for r in res)                       # the slowest process, without interpreter start-up
    return {"value": procs * n_hist * gens / busy, "unit": UNIT, "processes": procs, "cores_available": avail,
            "os_cpu_count": os.cpu_count(), "seconds": busy, "wall_seconds_with_startup": wall,
            "segments_per_sec": sum(r[1] for r in res) / busy}


def reference_arm(args):
    """--impl reference: the CPU oracle (single thread) on bounded samples of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    k = args.config
    n = args.oracle_n or (20_000 if EIG else 500_000 if DOGLEG else ORACLE_SAMPLE_N[k])
    gens = sum(EIG) if EIG else 1
    for _ in range(args.warmup and 1):
        run_oracle_sample(k, max(n // 10, 100))
    tot_t, tot_h, seg, fl = 0.0, 0, 0, 0
    for s in range(args.steps):
        dt, c = run_oracle_sample(k, n, seed=s)
        tot_t += dt; tot_h += n * gens; seg += c["segments"]; fl += c["flights"]
    val = tot_h / tot_t
    sample = f"config{k} with {n} histories per step (full geometry, tally and census schedule), single thread"
    if EIG:
        sample = f"the same cycles with {n} particles per cycle, single thread"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": workload_name(k, n)},
        "segments_per_sec": seg / tot_t, "flights_per_sec": fl / tot_t,
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--n-hist", type=int, default=0)
    ap.add_argument("--oracle-n", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-all-cores", action="store_true", help="skip the one-oracle-process-per-core baseline")
    ap.add_argument("--batches", type=int, default=0,
                    help="batches per step; 0 = as many as the library keeps in flight: 2 at the batch size of config 5, "
                         "8 for batches of at most 2e6 histories (configs 1-4, the eigenvalue pin cell)")
    ap.add_argument("--time-crossing", action="store_true",
                    help="switch the time-crossing block of the tally on (DESIGN.md C.13); the default workload has it off")
    ap.add_argument("--eigenvalue", default="", metavar="I,A",
                    help="run the pin-cell k-eigenvalue workload (DESIGN.md C.14) with I inactive and A active cycles "
                         "(the paper's run is 50,100 with --n-hist 100000) instead of a BASELINE.json config")
    ap.add_argument("--implicit-capture", default="", metavar="WR,WS",
                    help="switch implicit capture on (DESIGN.md C.15): roulette below WR back to WS, weighted comb; "
                         "the default workload is analog")
    ap.add_argument("--delayed", default="", metavar="BETA,TIME_SCALE",
                    help="add the seeded six-group delayed-neutron set (DESIGN.md C.16): delayed fraction BETA, decay "
                         "constants 0.0125..3 divided by TIME_SCALE seconds; the default workload is all prompt")
    ap.add_argument("--dogleg", type=int, default=0, metavar="SUB",
                    help="run the dog-leg void duct stand-in of the paper's time-dependent Kobayashi problem (source "
                         "window, DESIGN.md C.17; combine with --implicit-capture as the paper does) with SUB tally bins "
                         "per 10 cm cell and axis")
    ap.add_argument("--bank-factor", type=float, default=0.0,
                    help="bank_capacity_factor of mcdc_run (0 = the library default 1.5; implicit capture on a "
                         "supercritical config needs about 3: nobody is captured between census times)")
    ap.add_argument("--dump-steps", default="", help="write the per-census-step counters of the first timed batch to this JSON file")
    args = ap.parse_args()
    if args.implicit_capture:
        global IC
        IC = tuple(float(x) for x in args.implicit_capture.split(","))
    if args.dogleg:
        global DOGLEG
        DOGLEG = args.dogleg
        args.config = 2          # (sizes the oracle sample and the atomic-peak lookup only)
        args.n_hist = args.n_hist or 10_000_000
    if args.delayed:
        global DN
        DN = tuple(float(x) for x in args.delayed.split(","))
    if args.eigenvalue:
        global EIG
        EIG = tuple(int(x) for x in args.eigenvalue.split(","))
        args.config = 4          # (the closest BASELINE.json config: its materials and pin; sizes the atomic peak lookup)
        args.n_hist = args.n_hist or 100_000
    if args.impl == "reference":
        return reference_arm(args)

    import torch
    import torch.distributed as dist
    from paper_2305_07636_b200 import Problem

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    k = args.config
    n_hist = args.n_hist or FULL_N[k]
    cfg = make_cfg(k, n_hist)
    if args.time_crossing:
        cfg["tally"]["time_crossing"] = 1
    from paper_2305_07636_b200 import replicas
    prob = Problem(cfg)
    stream = torch.cuda.current_stream()
    nb = args.batches if args.batches > 0 else (8 if n_hist <= 2_000_000 else 2)

    # every rank runs its own batches: batch index = (step * world + rank) * nb + b -> Philox seed + index;
    # with N > 1 the replicas' sums and counters are all-reduced (NCCL, in place on the workspace) inside
    # the timed region, so that every rank ends the step holding the result of all N * nb batches
    def step(i, p=prob):
        p.run(seed=(i * world + rank) * nb, n_hist_per_batch=n_hist, n_batch=nb, stream=stream, bank_capacity_factor=args.bank_factor)
        if world > 1:
            replicas.combine(p)

    for i in range(args.warmup):
        step(1000 + i)
    barrier()
    clocks = ClockSampler(local) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    seg = fl = coll = launches = iters = 0
    kname = "k_pool" if prob.kernel_path() == "pool" else "k_flight"
    evb = 0
    if clocks:
        clocks.mark()
    e0.record(stream)
    for i in range(args.steps):
        step(i)
        for b in range(nb):
            c = prob.counters(b)      # (after combine: summed over the ranks)
            seg += c["segments"]; fl += c["flights"]; coll += c["collisions"]; evb += event_model_bytes(c)
        st = prob.stats(); launches += st["launches"]; iters += st["iterations"]
        if args.dump_steps and i == 0 and rank == 0:
            with open(args.dump_steps, "w") as f:
                json.dump([prob.counters(0, kk) for kk in range(prob.n_steps)], f)
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    k_eff = None
    if EIG:
        kc = prob.k_cycle(0)[EIG[0]:]
        k_eff = {"mean_active": float(kc.mean()), "std_of_mean": float(kc.std(ddof=1) / np.sqrt(len(kc))) if len(kc) > 1 else None,
                 "cycles": len(kc)}
    clk = clocks.stop() if clocks else None
    seg_ov, fl_ov = seg, fl
    # Per-launch kernel times for the roofline: CUDA events recorded by the library on the launching stream
    # around every launch of the event kernel (mcdc_profile).  They are taken on the same K steps repeated
    # with ONE batch in flight, because with several pipelines an event pair also spans the other
    # pipelines' kernels.  (Event timing makes the host wait for every launch, so it is kept out of the
    # timed region above.)
    prob.profile(True)
    kms = {kname: 0.0, "k_collide": 0.0}
    kln = {kname: 0, "k_collide": 0}
    fl = coll = seg = evb = 0
    ms_solo = 0.0
    for i in range(args.steps):
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record(stream)
        prob.run(seed=i * world + rank, n_hist_per_batch=n_hist, n_batch=1, stream=stream, bank_capacity_factor=args.bank_factor)
        a1.record(stream); torch.cuda.synchronize()
        ms_solo += a0.elapsed_time(a1)
        c = prob.counters(0)
        seg += c["segments"]; fl += c["flights"]; coll += c["collisions"]; evb += event_model_bytes(c)
        pr = prob.profile_read()
        for name in kms:
            kms[name] += pr[name]["ms"]; kln[name] += pr[name]["launches"]
    prob.profile(False)
    t = torch.tensor([ms], dtype=torch.float64, device="cuda")
    tot = torch.tensor([float(seg_ov), float(fl_ov)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)      # (the counters are already sums over the ranks)
    ms_all = float(t.item())
    hist_total = n_hist * nb * args.steps * world * (sum(EIG) if EIG else 1)
    value = hist_total / (ms_all * 1e-3)

    # end to end through the public API with HOST buffers, every step: problem tables host->device (create),
    # run (+ combine), mean and standard error of the tally + counters device->host into pinned memory,
    # destroy.  The device workspace and the pinned buffer are caller-owned and reused.
    e2e = None
    if not args.no_e2e:
        h2d = sum(int(np.asarray(v).nbytes) for grp in ("materials", "geometry", "tally") for v in cfg[grp].values()
                  if hasattr(v, "nbytes"))
        n_read = 2 if nb * world >= 2 else 1
        d2h = int(np.prod(prob.shape)) * 8 * n_read + 16 * 8 * prob.n_steps * nb
        ws_keep = prob._ws
        pins = [torch.empty(int(np.prod(prob.shape)), dtype=torch.float64, pin_memory=True) for _ in range(n_read)]
        parts = {"create_ms": 0.0, "run_ms": 0.0, "read_ms": 0.0, "destroy_ms": 0.0}
        barrier()
        t0 = time.perf_counter()
        for i in range(args.steps):
            ta = time.perf_counter()
            p2 = Problem(cfg)
            p2._ws = ws_keep                      # device workspace is caller-owned and reused
            tb = time.perf_counter()
            step(i, p2)
            tc = time.perf_counter()
            chk = 0.0
            for w in range(n_read):
                p2._pin = pins[w]
                out = p2.tally(w, pinned=True)
                chk += float(out[0].sum())
            _ = [p2.counters(b) for b in range(nb)]
            td_ = time.perf_counter()
            p2._ws = None; p2._pin = None
            p2.close()
            te = time.perf_counter()
            parts["create_ms"] += 1e3 * (tb - ta); parts["run_ms"] += 1e3 * (tc - tb)
            parts["read_ms"] += 1e3 * (td_ - tc); parts["destroy_ms"] += 1e3 * (te - td_)
        barrier()
        dt = time.perf_counter() - t0
        td = torch.tensor([dt], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(td, op=dist.ReduceOp.MAX)
        e2e = {"value": hist_total / float(td.item()), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "reads": "mean" + (" + standard error" if n_read == 2 else "") + " + counters",
               "ms_per_step": {k2: v / args.steps for k2, v in parts.items()}, "checksum": chk}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # Roofline of the dominant kernel.  The metric is "% of HBM/atomic roofline" (BASELINE.json): the
    # headline fraction is SURVEY 8(d)'s algorithmic bytes of the events the kernel processed / its
    # CUDA-event time, against the measured HBM copy bandwidth.  Beside it: the bytes the kernel really
    # moves (`traffic`, ncu), the issue-slot utilisation that actually limits it, and the tally REDs
    # against the measured fp64 atomic peak (ncu counters per segment x the run's segments).
    peak, peak_src = measured_peak_hbm()
    kt = kms[kname] * 1e-3
    cal_path = next((os.path.join(ROOT, "profiles", f) for f in ("pool_r2.json", "pool_r1.json")
                     if os.path.exists(os.path.join(ROOT, "profiles", f))), None)
    wl = "dogleg" if DOGLEG else "eigenvalue" if EIG else f"config{k}"
    if kname == "k_pool":
        with open(cal_path) as f:
            cal_all = json.load(f)
        cal = cal_all.get(wl) or cal_all.get("config5") or cal_all
        ipeak, ipeak_src = issue_peak()
        ach = cal["warp_inst_per_flight"] * fl / kt / 1e9 if kt > 0 else 0.0
        hbm_ach = evb / kt / 1e9 if kt > 0 else 0.0
        roofline = {"bound": "hbm", "kernel": kname, "achieved": hbm_ach, "peak": peak, "unit": "GB/s",
                    "frac": hbm_ach / peak, "traffic": cal["dram_bytes_per_flight"] * fl / max(kln[kname], 1),
                    "peak_source": peak_src, "algorithmic_bytes": EVENT_MODEL,
                    "algorithmic_bytes_per_launch": evb / max(kln[kname], 1),
                    "flights_per_launch": fl / max(kln[kname], 1),
                    "avg_launch_ms": kms[kname] / max(kln[kname], 1),
                    "share_of_step": {n: kms[n] / ms_solo for n in kms},
                    "measured_on": "the same K steps with one batch in flight (un-overlapped launches), CUDA events on the launching stream",
                    "note": "algorithmic = the bytes the per-event-kernel form moves for the events this kernel processed "
                            "(SURVEY 8(d)); the kernel keeps particles on chip and moves only `traffic` (ncu), so this fraction "
                            "is a work rate on the north_star's yardstick, not DRAM utilisation; the resource that limits "
                            "the kernel is instruction issue (`issue_slots`)",
                    "issue_slots": {"achieved": ach, "peak": ipeak, "unit": "Gwarp-inst/s", "frac": ach / ipeak,
                                    "peak_source": ipeak_src,
                                    "per_unit": {"warp_inst_per_flight": cal["warp_inst_per_flight"], "source": cal["source"]}}}
    else:
        bytes_move = fl * 120 + (fl - coll) * 16 + seg * 8
        achieved = bytes_move / kt / 1e9 if kt > 0 else 0.0
        roofline = {"bound": "hbm", "kernel": kname, "achieved": achieved, "peak": peak, "unit": "GB/s",
                    "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": bytes_move / max(kln[kname], 1),
                    "avg_launch_ms": kms[kname] / max(kln[kname], 1),
                    "share_of_step": {n: kms[n] / ms_solo for n in kms},
                    "measured_on": "the same K steps with one batch in flight (un-overlapped launches)"}
        tr = os.path.join(ROOT, "profiles", "traffic.json")
        if os.path.exists(tr):
            with open(tr) as f:
                roofline["traffic"] = json.load(f).get("k_flight_dram_bytes_per_launch")
    ap = os.path.join(ROOT, "profiles", "atomic_peak_r2.json")
    if os.path.exists(ap) and kname == "k_pool" and "red_sectors_per_segment" in cal:
        # tally REDs in L2 reduction sectors (ncu lts__t_sectors_op_red.sum): achieved = the
        # committed capture's sectors per scored segment of this workload x this run's segments / kernel time; peak =
        # the measured fp64 atomic rate x its sectors per atomic, for the array size the step keeps hot
        with open(ap) as f:
            pk = json.load(f)
        peaks = {int(k2): v for k2, v in pk["red_sectors_per_s_by_bins"].items()}
        hot = max(1, int(np.prod(prob.shape)) // max(1, prob.n_steps if not EIG else 1))   # bins one census step can touch
        key = min(peaks, key=lambda b: abs(np.log(b) - np.log(max(hot, 1))))
        red_rate = cal["red_sectors_per_segment"] * seg / kt if kt > 0 else 0.0
        roofline["atomic"] = {"achieved": red_rate, "peak": peaks[key], "unit": "L2 RED sectors/s",
                              "frac": red_rate / peaks[key], "hot_bins": hot, "peak_measured_at_bins": key,
                              "red_sectors_per_segment": cal["red_sectors_per_segment"],
                              "note": "profiles/pool_r2.json (ncu capture of this workload) and profiles/atomic_peak_r2.md"}
    cpu = None
    if not args.no_cpu_baseline:
        n_o = args.oracle_n or (20_000 if EIG else 500_000 if DOGLEG else ORACLE_SAMPLE_N[k])
        dt, c = run_oracle_sample(k, n_o)
        cpu = {"value": n_o * (sum(EIG) if EIG else 1) / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": (f"the same cycles with {n_o} particles per cycle, {dt:.1f} s" if EIG else
                          f"{wl} with {n_o} histories (full geometry, tally and census schedule), {dt:.1f} s"),
               "segments_per_sec": c["segments"] / dt}
        if not args.no_all_cores:
            cpu["all_cores"] = run_oracle_all_cores(k, n_o)
            cpu["cores_available"] = cpu["all_cores"]["cores_available"]

    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_all / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(k, n_hist) + f" x {nb} batches per step" +
                   (" + time-crossing tally block" if args.time_crossing else "") +
                   (f"; {world} replicas, sums and counters all-reduced every step" if world > 1 else ""),
                   "l2": "working set (particle banks 0.8 GB + 294 MB tally) larger than L2; no flush needed"
                   if k >= 4 and not EIG else "working set fits L2: launch/atomic-bound, see DESIGN.md"},
        "segments_per_sec": float(tot[0].item()) / (ms_all * 1e-3),
        "flights_per_sec": float(tot[1].item()) / (ms_all * 1e-3),
        "gpu_launches": launches, "event_iterations": iters, **({"k_eff": k_eff} if EIG else {}),
        "clocks": clk, "e2e": e2e, "roofline": roofline, "cpu_baseline": cpu,
    }))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
