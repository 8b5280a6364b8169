#!/usr/bin/env python
"""bench.py -- fitted tracks/s of the batched Kalman track fit on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one pass of the whole hot path (forward filter + RTS smoother = one kf_fit_batch
call) over one batch of synthetic tracks.  Default workload: BASELINE.json configs[2]
(1,000,000 tracks x 30 layers with material, filter + smoother, seed 3) -- the configuration the
north_star target is quoted on.  Inputs are resident in HBM for `value`; `e2e` goes through
kf_fit_batch_host with pinned HOST buffers (H2D + fit + D2H inside the timed region).

The path does not shard (north_star: one GPU, no collectives): with --gpus N > 1 (under torchrun)
every rank fits its own replica of the batch ("replicas only"); value is
the tracks all ranks fitted / max-over-ranks time.

--impl reference times the CPU oracle (oracle/, as it stands) on the box's host cores on a
bounded sample of the same workload.
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

METRIC = "fitted tracks/sec (device-timed, FP64)"
UNIT = "tracks/s"

# Work per leg (one surface visited by one track), DESIGN.md "Rooflines".
#   bytes: RTS record 55 doubles + 1 flag byte written by the forward kernel and read by the RTS
#          kernel, the hit (2 doubles + int32) read by both; per track 27 doubles in, outputs out.
#   flops, two clearly separate counts (DFMA = 2, DMUL/DADD = 1):
#     ALGORITHMIC  SURVEY.md 8(d) D.3: the hand count of the method as stated (dense 3x3 stage chains, three
#                  RKN4 steps, library transcendentals as FP64-instruction equivalents).  A property of the method.
#     EXECUTED     what the kernels issue, from the opcode table of the committed ncu capture named below
#                  (warp-level DFMA/DMUL/DADD of one launch x 32 / legs of that launch).  The closed-form
#                  constant-field step and the structured products make it 1.8x smaller than the hand count, so
#                  only THIS count may be divided by a measured FP64 peak.  FP64_PIPE = FP64-pipe instructions
#                  (DFMA + DMUL + DADD + DSETP) per leg and thread from the same table: the issue-slot view.
REC_BYTES = 55 * 8 + 1
HIT_BYTES = 2 * 8 + 4
ALGORITHMIC_FLOP_PER_LEG = dict(source="SURVEY.md 8(d) D.3 (hand count of the method)",
                                forward={"const": 3450.0, "const_nomat": 3200.0, "grid3": 4000.0}, rts=1650.0 + 170.0)
# What the committed ncu capture says (profiles/r03_cfg2_ncu_summary.md; tests/test_bench_contract.py re-reads the file and
# fails when these numbers and its tables differ): warp-level instruction counts in millions per launch from the opcode
# table, DRAM Gbyte (read, write) and the FP64-pipe percentage from the counter table; one launch = 262,144 tracks x 30 legs.
CAPTURE_COUNTS = dict(
    source="profiles/r03_cfg2_ncu_summary.md", legs=262144 * 30,
    opcodes_M=dict(kf_forward_kernel=dict(DFMA=172.182, DMUL=78.822, DADD=22.845, DSETP=7.386),
                   kf_rts_kernel=dict(DFMA=183.738, DMUL=44.556, DADD=14.057, DSETP=3.817)),
    dram_gbyte=dict(kf_forward_kernel=(0.251638, 3.624636), kf_rts_kernel=(3.474265, 0.056504)),
    fp64_pipe_pct=dict(kf_forward_kernel=61.9, kf_rts_kernel=61.5))


def _per_leg(kernel, ops, weight):
    c = CAPTURE_COUNTS["opcodes_M"][kernel]
    return sum(c[o] * w for o, w in zip(ops, weight)) * 1e6 * 32 / CAPTURE_COUNTS["legs"]


EXECUTED_PER_LEG = dict(source=CAPTURE_COUNTS["source"] + " (opcode table; 262,144 tracks x 30 legs = 7,864,320 legs per launch)",
                        flop={k: _per_leg(k, ("DFMA", "DMUL", "DADD"), (2, 1, 1)) for k in ("kf_forward_kernel", "kf_rts_kernel")},
                        fp64_pipe_instr={k: _per_leg(k, ("DFMA", "DMUL", "DADD", "DSETP"), (1, 1, 1, 1))
                                         for k in ("kf_forward_kernel", "kf_rts_kernel")},
                        fp64_pipe_pct_ncu=dict(CAPTURE_COUNTS["fp64_pipe_pct"]),
                        workload="cfg2 (constant field, material, RTS)")
# The executed counts and the DRAM traffic belong to the kernels as they were when the capture was taken: the hash of
# csrc/ at that commit is kept here, and a library built from other sources (or with tuning -D macros, or another
# instantiation than the captured one) gets null instead of a stale fraction (kernel_sources_sha16 below).
CAPTURE = dict(sources_sha16="0ee0547f726f85a4", commit="the commit that adds profiles/r03_cfg2_ncu_summary.md",
               instantiation="kf_forward_kernel<FIELD_CONST, MATERIAL, GEOM_SMEM, 1, 256, 0, PLAIN, double, 0> + kf_rts_kernel<PLAIN, double>: "
                             "cfg2, more than 37,888 tracks, minimal outputs, default stepping, default build")
FP64_LANES_PER_SM = 64  # FP64 FMA lanes per SM on B200 (148 SMs x 64 x 2 flop x clock)
# DRAM traffic per leg measured by ncu --set full (dram__bytes_read.sum + dram__bytes_write.sum of one launch
# over 262,144 tracks x 30 legs of this workload, divided by the legs), from the committed capture below.
# bench.py scales it to the launch it times; it is not re-measured live (never time under a profiler).
NCU_TRAFFIC = dict(source=CAPTURE_COUNTS["source"],
                   bytes_per_leg={k: sum(v) * 1e9 / CAPTURE_COUNTS["legs"] for k, v in CAPTURE_COUNTS["dram_gbyte"].items()})


def kernel_sources_sha16():
    """sha256 (first 16 hex digits) over the names and contents of csrc/*.cu, *.cuh, *.h: what the kernels are built from"""
    import hashlib
    from paper_2105_01796_b200 import build as kbuild
    h = hashlib.sha256()
    for path in kbuild.sources() + [q for q in kbuild.headers() if os.path.dirname(q) == kbuild.CSRC]:
        h.update(os.path.basename(path).encode())
        with open(path, "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2,
                    help="BASELINE.json configs index (default 2); 5 / 6: the barrel / endcap workloads of the cylinder and "
                         "disc surface kinds (context, not BASELINE configs)")
    ap.add_argument("--tracks", type=int, default=None, help="override the number of tracks (testing)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--variant", default="auto", choices=["auto", "thread", "lanes"],
                    help="kernel variant (kf_options.variant): thread per track or 8 lanes per track")
    ap.add_argument("--smoother", default="rts", choices=["rts", "bf"],
                    help="backward pass (kf_options.smoother): Rauch-Tung-Striebel (default, the north_star's) or the "
                         "Bryson-Frazier form of the same smoothed state (42-double records, no 6x6 solve)")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "mixed"],
                    help="arithmetic (kf_options.precision): fp64 = the BASELINE.json metric (default); mixed = the paper's "
                         "operating point, float operands and records with the 6x6 solve in double (PAPER.md:160-164, 272)")
    ap.add_argument("--field-stage", action="store_true",
                    help="grid field: pass the shared-memory staging hint (kf_field.stage_*, kf_field_stage_box): the acceptance "
                         "box of the table is kept in shared memory instead of being read through L1/L2 (measured slower on cfg4)")
    ap.add_argument("--field-gradient", action="store_true",
                    help="grid field: carry the dB/dr terms in the transported Jacobian (kf_options.field_gradient; the "
                         "general kernels)")
    ap.add_argument("--perigee", action="store_true",
                    help="also extrapolate the result to the perigee surface (the z axis through the origin): one more kernel "
                         "per step (kf_perigee_kernel); context runs and ncu captures, not the bench line")
    ap.add_argument("--mode", default="batch", choices=["batch", "events", "pcie", "resolution"],
                    help="batch (default): the bench line, one kf_fit_batch call over the whole workload per step.  "
                         "events: the same workload cut into --events calls of equal size (event-at-a-time, SURVEY 8(f) #4; "
                         "BASELINE configs[3]: 100 events x 10,000 tracks), issued round-robin on --streams streams, or all "
                         "captured once in a CUDA graph (--graph) and replayed; one context line.  pcie: pinned-memory copy "
                         "rates of this box (H2D alone, D2H alone, both at once): the floor of the e2e number; one context line.  "
                         "resolution: the MIXED-precision fit against the FP64 fit of the same batch (both through the "
                         "library): shifts of the fitted parameters in standard deviations, variances, chi2; one context line")
    ap.add_argument("--events", type=int, default=100)
    ap.add_argument("--streams", type=int, default=1)
    ap.add_argument("--graph", action="store_true")
    ap.add_argument("--e2e-chunk", type=int, default=65536, help="tracks per chunk of the pipelined host call (e2e)")
    ap.add_argument("--e2e-streams", type=int, default=3, help="streams of the pipelined host call (e2e)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-alt-precision", action="store_true", help="skip the MIXED-precision context key of the FP64 line")
    return ap.parse_args()


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(hbm_gbs=float(p["hbm_gbs"]), sm_max_mhz=float(p.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [l for (t, l) in self.lines if t0 - 0.2 <= t <= t1 + 0.3] or [l for (_, l) in self.lines]
        for l in rows:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for nme, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(smax) if smax else None,
                    power_w=float(np.median(power)) if power else None, samples=len(sm), reasons=sorted(reasons))


def dist_setup(n_gpus):
    """-> (rank, world, dist or None). Under torchrun the env carries RANK/WORLD_SIZE/LOCAL_RANK."""
    from paper_2105_01796_b200 import replicas
    rank, local, world = replicas.rank_world()
    if world > 1:
        import torch
        torch.cuda.set_device(local)
        return rank, world, replicas.init("nccl")
    return 0, 1, None


def cpu_baseline(wl, cores_hint=None):
    """The oracle as it stands on a bounded sample (first tracks of the same workload): all host cores (OpenMP over
    tracks, the paper's CPU parallelisation) and, beside it, one thread.  A short
    probe sets the samples so that each of the three timed runs per figure is about 5 s / 2 s of wall clock (capped at the
    workload); the best of the three is reported, all three are kept."""
    import oracle  # test infrastructure; bench.py's cpu_baseline leg is one of its allowed callers
    n0 = int(min(wl.n_tracks, 20_000))
    oracle.fit_workload(wl.subset(np.arange(min(64, n0))))  # builds/loads the library outside the timing
    t = time.perf_counter()
    oracle.fit_workload(wl.subset(np.arange(n0)))
    rate = n0 / max(time.perf_counter() - t, 1e-6)
    n = int(min(wl.n_tracks, max(n0, rate * 5.0)))
    sub = wl.subset(np.arange(n))
    # wall clock, best of 3 (all three kept in `runs_s`)
    runs = []
    for _ in range(3):
        t = time.perf_counter()
        r = oracle.fit_workload(sub)
        runs.append(time.perf_counter() - t)
    dt = min(runs)
    cores = int(r.threads)
    n1 = int(min(n, max(2000, rate / max(cores, 1) * 2.0)))
    sub1 = wl.subset(np.arange(n1))
    runs1 = []
    for _ in range(3):
        t = time.perf_counter()
        r1 = oracle.fit_workload(sub1, n_threads=1)
        runs1.append(time.perf_counter() - t)
    dt1 = min(runs1)
    assert int(r1.threads) == 1
    return dict(value=n / dt, unit=UNIT, cores=cores, kind="oracle",
                sample=f"first {n} tracks of {wl.name} ({sub.n_meas} hits), best of 3 runs: {dt:.2f} s wall, OpenMP over tracks",
                runs_s=[round(v, 4) for v in runs],
                one_thread=dict(value=n1 / dt1, unit=UNIT, cores=1, runs_s=[round(v, 4) for v in runs1],
                                sample=f"first {n1} tracks of {wl.name}, best of 3 runs: {dt1:.2f} s wall, 1 thread"))


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, K steps of a bounded sample each."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    from paper_2105_01796_b200 import workloads as W
    cores = os.cpu_count() or 1
    n = int(min(args.tracks or 10**9, 1500 * cores, 100_000))
    wl = W.make_workload(args.config, n_tracks=n)
    for _ in range(max(args.warmup, 1)):
        r = oracle.fit_workload(wl)
    t = time.perf_counter()
    for _ in range(args.steps):
        r = oracle.fit_workload(wl)
    dt = (time.perf_counter() - t) / args.steps
    val = n / dt
    line = dict(impl="reference", metric=METRIC, value=val, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=dt * 1e3, higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=W.WORKLOAD_NAMES[args.config], tracks_per_step=n,
                            note="CPU oracle on a bounded sample of the workload (seeded generator, first tracks)"),
                cpu_baseline=dict(value=val, unit=UNIT, cores=int(r.threads), kind="oracle",
                                  sample=f"{n} tracks of cfg{args.config} per step"),
                e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                gpu_launches=0)
    print(json.dumps(line))
    return 0


def run_events(args):
    """Event-at-a-time (U20): the workload as --events independent kf_fit_batch calls
    (resident inputs, one workspace and one output set per stream so that calls on different streams do not share
    scratch), CUDA events around all of them; --graph: the calls of one step captured once, the graph replayed."""
    import torch
    import paper_2105_01796_b200 as kf
    from paper_2105_01796_b200 import workloads as W
    dev = torch.device("cuda", 0)
    wl = W.make_workload(args.config, n_tracks=args.tracks)
    n_ev = args.events
    per = wl.n_tracks // n_ev
    assert per > 0
    S = 1 if args.graph else max(1, args.streams)
    calls = []
    for e in range(n_ev):
        sub = wl.subset(np.arange(e * per, (e + 1) * per))
        hb = kf.HostBatch.from_workload(sub)
        db = kf.DeviceBatch(hb, dev)
        calls.append((db, hb))
    # one output set + workspace per stream slot (calls on one stream run in order and may share them)
    outs = [kf.DeviceOutputs(per, max(hb.n_meas for _, hb in calls), calls[0][1].n_legs_max, 0, per_hit=True, rk_err=False,
                             device=dev) for _ in range(S)]
    fits = []
    for e, (db, hb) in enumerate(calls):
        out = kf.DeviceOutputs(per, hb.n_meas, hb.n_legs_max, 0, per_hit=True, rk_err=False, device=dev) if args.graph or S > 1 else outs[0]
        fits.append(kf.FitCall(db, out=out))
    streams = [torch.cuda.Stream(dev) for _ in range(S)]

    def issue():
        for e, f in enumerate(fits):
            f.run(stream=streams[e % S])

    main_stream = torch.cuda.current_stream(dev)

    def step_plain():
        for st in streams:
            st.wait_stream(main_stream)
        issue()
        for st in streams:
            main_stream.wait_stream(st)

    graph = None
    if args.graph:
        for _ in range(3):
            step_plain()
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        cap = torch.cuda.Stream(dev)
        with torch.cuda.graph(graph, stream=cap):
            for f in fits:
                f.run(stream=torch.cuda.current_stream(dev))
        step = graph.replay
    else:
        step = step_plain
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    for k in range(args.steps):
        ev[k].record()
        step()
    ev[args.steps].record()
    torch.cuda.synchronize()
    per_step = np.array([ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)])
    launches = sum(f.launches for f in fits)
    print(json.dumps(dict(mode="events", metric=METRIC, unit=UNIT, value=per * n_ev / (per_step.mean() * 1e-3),
                          ms_per_step=float(per_step.mean()), median_ms=float(np.median(per_step)), steps=args.steps,
                          config=dict(workload=W.WORKLOAD_NAMES[args.config], events=n_ev, tracks_per_event=per,
                                      streams=S, cuda_graph=bool(args.graph)),
                          ms_per_event=float(per_step.mean() / n_ev), gpu_launches=launches * args.steps,
                          note="context line (event-at-a-time regime), not the bench line")))
    return 0


def run_pcie(args):
    """Pinned-memory copy rates of this box with plain torch copies of the sizes the e2e call moves (820 MB in, 460 MB
    out per 1e6-track CFG2 call): each direction alone and both at once on two streams."""
    import torch
    dev = torch.device("cuda", 0)
    n_in, n_out = 820_000_000, 460_000_000
    h_in = torch.empty(n_in, dtype=torch.uint8).pin_memory()
    h_out = torch.empty(n_out, dtype=torch.uint8).pin_memory()
    d_in = torch.empty(n_in, dtype=torch.uint8, device=dev)
    d_out = torch.empty(n_out, dtype=torch.uint8, device=dev)
    s1, s2 = torch.cuda.Stream(dev), torch.cuda.Stream(dev)

    def timed(fn, reps=5):
        fn()
        torch.cuda.synchronize()
        t = []
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            t.append(e0.elapsed_time(e1))
        return float(np.median(t))

    def h2d():
        d_in.copy_(h_in, non_blocking=True)

    def d2h():
        h_out.copy_(d_out, non_blocking=True)

    def both():
        cur = torch.cuda.current_stream(dev)
        s1.wait_stream(cur)
        s2.wait_stream(cur)
        with torch.cuda.stream(s1):
            d_in.copy_(h_in, non_blocking=True)
        with torch.cuda.stream(s2):
            h_out.copy_(d_out, non_blocking=True)
        cur.wait_stream(s1)
        cur.wait_stream(s2)

    t_in, t_out, t_both = timed(h2d), timed(d2h), timed(both)
    print(json.dumps(dict(mode="pcie", h2d_bytes=n_in, d2h_bytes=n_out, h2d_ms=t_in, d2h_ms=t_out, both_ms=t_both,
                          h2d_gbs=n_in / t_in / 1e6, d2h_gbs=n_out / t_out / 1e6,
                          both_total_gbs=(n_in + n_out) / t_both / 1e6,
                          note="context line: plain pinned copies, no library call; the e2e number's floor is both_ms")))
    return 0


def run_resolution(args):
    """PAPER.md:314-318 (float against double): the MIXED fit (float operands and records, 6x6 solve in double) against the
    FP64 fit of the same batch, both by the library: |dx| / sigma of the fitted parameters (first_* and last_*), relative
    change of their variances, |dchi2|, discrete decisions that differ; and the time of both."""
    import torch
    import paper_2105_01796_b200 as kf
    from paper_2105_01796_b200 import workloads as W
    dev = torch.device("cuda", 0)
    wl = W.make_config(args.config, n_tracks=args.tracks or 200_000)
    hb = kf.HostBatch.from_workload(wl)
    db = kf.DeviceBatch(hb, dev)
    res, ms = {}, {}
    for name, prec in (("fp64", 0), ("mixed", 1)):
        call = kf.FitCall(db, precision=prec)
        for _ in range(3):
            call.run()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            call.run()
        e1.record()
        torch.cuda.synchronize()
        ms[name] = e0.elapsed_time(e1) / args.steps
        res[name] = call.out.to_host()
    a, b = res["fp64"], res["mixed"]
    same = (a.status == b.status) & (a.n_used == b.n_used) & (a.n_outliers == b.n_outliers)
    ok = same & ((a.status & 7) == 0)
    out = dict(mode="resolution", config=dict(workload=W.WORKLOAD_NAMES[args.config], tracks=int(wl.n_tracks)),
               tracks_compared=int(ok.sum()), tracks_with_a_different_decision=int((~same).sum()),
               ms_fp64=ms["fp64"], ms_mixed=ms["mixed"])
    names = ["loc0", "loc1", "phi", "theta", "qp", "t"]
    for nm in ("first", "last"):
        va = np.einsum("nii->ni", getattr(a, nm + "_cov"))[ok]
        vb = np.einsum("nii->ni", getattr(b, nm + "_cov"))[ok]
        d = (getattr(b, nm + "_params") - getattr(a, nm + "_params"))[ok]
        d[:, 2] = (d[:, 2] + np.pi) % (2 * np.pi) - np.pi
        z = np.abs(d) / np.sqrt(va)
        out[nm] = dict(rms_sigma={n_: float(v) for n_, v in zip(names, np.sqrt(np.mean(z ** 2, axis=0)))},
                       max_sigma={n_: float(v) for n_, v in zip(names, z.max(axis=0))},
                       max_var_rel=float(np.max(np.abs(vb / va - 1.0))))
    out["max_abs_dchi2"] = float(np.max(np.abs(a.chi2 - b.chi2)[ok]))
    out["mean_chi2"] = dict(fp64=float(a.chi2[ok].mean()), mixed=float(b.chi2[ok].mean()))
    print(json.dumps(out))
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.mode == "resolution":
        return run_resolution(args)
    if args.mode == "events":
        return run_events(args)
    if args.mode == "pcie":
        return run_pcie(args)

    import torch
    import paper_2105_01796_b200 as kf
    from paper_2105_01796_b200 import binding as B
    from paper_2105_01796_b200 import replicas
    from paper_2105_01796_b200 import workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the fit has no CPU fallback")
    rank, world, dist = dist_setup(args.gpus)
    dev = torch.device("cuda", torch.cuda.current_device())
    peaks = load_peaks()

    wl = W.make_workload(args.config, n_tracks=args.tracks)
    hb = kf.HostBatch.from_workload(wl)
    db = kf.DeviceBatch(hb, dev)
    variant = {"auto": 0, "thread": 1, "lanes": 2}[args.variant]
    bf = args.smoother == "bf"
    # minimal outputs: first/last state, chi2, ndf, status, counters, per-hit chi2 and flags (no RKN error diagnostic)
    out = kf.DeviceOutputs(hb.n_tracks, hb.n_meas, hb.n_legs_max, 0, per_hit=True, rk_err=False, device=dev)
    mixed = args.precision == "mixed"
    if args.perigee:
        out = kf.DeviceOutputs(hb.n_tracks, hb.n_meas, hb.n_legs_max, 0, per_hit=True, rk_err=False, device=dev, perigee=True)
    call = kf.FitCall(db, out=out, variant=variant, smoother=int(bf), precision=int(mixed),
                      field_stage=args.field_stage, field_gradient=int(args.field_gradient),
                      perigee=((0.0, 0.0, 0.0), (0.0, 0.0, 1.0)) if args.perigee else None)
    N, M = hb.n_tracks, hb.n_meas
    smooth = bool(hb.options.get("smooth", 1))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    t_warm = time.time()
    for _ in range(max(args.warmup, 3)):
        call.run()
    barrier()
    # a fresh box ramps its clocks over the first few hundred milliseconds of load (a cold first run measured 1916 MHz
    # and 6.0 ms per step against 1965 MHz and 5.8 ms): keep warming up, untimed, until half a second has passed
    extra_warmup = 0
    while time.time() - t_warm < 0.5 and extra_warmup < 200:
        call.run()
        extra_warmup += 1
        if extra_warmup % 8 == 0:
            torch.cuda.synchronize()
    barrier()
    fp64_probe = kf.probe_fp64_tflops(20000, dev) if rank == 0 else None

    # ---- timed region: exactly K steps, CUDA events on the launching stream ----------------------------
    timer = B.StageTimer(dev)
    timer.prepare(args.steps)
    sampler = ClockSampler(dev.index or 0)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    barrier()
    # one event before every step and one after the last: the whole region (value) and every step (statistics)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    t_wall0 = time.time()
    for k in range(args.steps):
        ev[k].record()
        timer.arm(k)
        call.run()
    ev[args.steps].record()
    barrier()
    t_wall1 = time.time()
    fwd_ms, rts_ms = timer.finish()
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    value, ms_total, n_job = replicas.job_throughput(N * args.steps, ev[0].elapsed_time(ev[args.steps]), dist, dev)
    ms_step = ms_total / args.steps
    # SURVEY.md 8(d) D.4 / PAPER.md:268: median, and the paper-style mean +- RMS deviation over the timed calls (this rank)
    per_step = np.array([ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)])
    step_stats = dict(n=int(per_step.size), median_ms=float(np.median(per_step)), mean_ms=float(per_step.mean()),
                      rms_ms=float(np.sqrt(np.mean((per_step - per_step.mean()) ** 2))),
                      min_ms=float(per_step.min()), max_ms=float(per_step.max()),
                      note="per-step CUDA-event times on the launching stream; rms = sqrt(mean squared deviation) as PAPER.md:268")
    launches = call.launches * args.steps

    # results of the last step, for the legs count and a sanity line
    res = call.out
    n_legs = int((res.n_used.sum() + res.n_outliers.sum() + res.n_holes.sum()).item())
    bad = int(((res.status & 7) != 0).sum().item())

    # ---- end to end through the HOST-buffer entry point -------------------------------------------------
    e2e = None
    if not args.no_e2e:
        def time_host(hc):
            for _ in range(2):
                hc.run()
            barrier()
            h0, h1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ke = max(3, min(args.steps, 5))
            h0.record()
            for _ in range(ke):
                hc.run()
            h1.record()
            barrier()
            return replicas.max_over_ranks(h0.elapsed_time(h1), dist, dev) / ke, ke
        # the public host-buffer call: chunks of whole CTAs over a few streams (H2D, fit and D2H of different chunks overlap)
        hc = kf.HostCall(hb, dev, n_streams=args.e2e_streams, chunk_tracks=args.e2e_chunk, smoother=int(bf), precision=int(mixed),
                         field_stage=args.field_stage)
        ms_e2e, ke = time_host(hc)
        e2e = dict(value=world * N / (ms_e2e * 1e-3), unit=UNIT, h2d_bytes_per_step=int(hc.h2d_bytes),
                   d2h_bytes_per_step=int(hc.d2h_bytes), ms_per_step=ms_e2e, steps=ke, launches_per_step=int(hc.launches),
                   api=f"kf_fit_batch_host_pipelined (pinned host buffers; chunks of {args.e2e_chunk} tracks on {args.e2e_streams} streams: "
                       "H2D, forward, RTS, D2H per chunk)")
        del hc
        hc = kf.HostCall(hb, dev, smoother=int(bf), precision=int(mixed), field_stage=args.field_stage)  # context: the same through kf_fit_batch_host, everything in order on one stream
        ms_one, _ = time_host(hc)
        e2e["single_stream_ms_per_step"] = ms_one
        del hc

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- rooflines -------------------------------------------------------------------------------------
    fwd = float(np.mean(fwd_ms))
    rts = float(np.mean(rts_ms)) if smooth else 0.0
    fkind = hb.field_kind
    rec_b = (42 * 8 if bf else (55 * 4 + 1 if mixed else REC_BYTES)) if smooth else 0   # Bryson-Frazier record: 42 doubles, no flag byte; MIXED: 55 floats
    fwd_bytes = n_legs * rec_b + M * HIT_BYTES + N * (27 * 8 + 8) + N * (2 * 27 * 8 + 8 + 5 * 4) + M * 9
    rts_bytes = n_legs * rec_b + M * HIT_BYTES + N * (27 * 8 + 12)
    if bf:  # no hits re-read; the first-leg block (27 doubles) read, first_* written
        rts_bytes = n_legs * rec_b + N * (27 * 8 + 27 * 8 + 8)
        fwd_bytes += N * 27 * 8
    material = int(hb.options.get("material", 0))
    akey = "grid3" if fkind == "grid3" else ("const" if material else "const_nomat")
    alg = dict(kf_forward_kernel=ALGORITHMIC_FLOP_PER_LEG["forward"][akey], kf_rts_kernel=ALGORITHMIC_FLOP_PER_LEG["rts"])
    # the executed counts are of the capture's workload (constant field, material, RTS); other configs: null
    # ... and of the captured instantiation (PLAIN, 256-thread CTA: cfg2 itself above 37,888 tracks, minimal outputs,
    # default stepping), built from the captured sources without tuning macros; anything else: null, with the reason
    from paper_2105_01796_b200 import build as kbuild
    why_not = []
    if not (fkind == "const" and material == 1 and smooth and not bf and not mixed and args.config == 2):
        why_not.append("another workload or option set than the capture's (cfg2, FP64, RTS)")
    if not (N > 148 * 2 * 128 and variant != 2):
        why_not.append("another instantiation than the capture's (small-batch CTA or lanes variant)")
    if kbuild.built_defines():
        why_not.append("library built with tuning macros " + " ".join(kbuild.built_defines()))
    sha = kernel_sources_sha16()
    if sha != CAPTURE["sources_sha16"]:
        why_not.append(f"csrc/ changed since the capture (sha16 {sha} != {CAPTURE['sources_sha16']}): refresh "
                       + EXECUTED_PER_LEG["source"].split(" ")[0])
    exe_ok = not why_not
    fp64_nominal = 148 * FP64_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12  # TFLOP/s at max clock
    fp64_peak = float(fp64_probe)   # the DFMA-chain probe of THIS run (same box, same clocks, same power cap)
    hbm_peak = peaks["hbm_gbs"]

    def kernel_roof(name, key, ms, nbytes):
        if ms <= 0:
            return None
        sec = ms * 1e-3
        k = dict(kernel=name, ms=ms, hbm_gbs=nbytes / sec / 1e9, hbm_frac=nbytes / sec / 1e9 / hbm_peak,
                 algorithmic_flop_per_leg=alg[key], algorithmic_tflops=alg[key] * n_legs / sec / 1e12)
        if exe_ok:
            ex = EXECUTED_PER_LEG["flop"][key] * n_legs / sec / 1e12
            k.update(executed_flop_per_leg=EXECUTED_PER_LEG["flop"][key], executed_tflops=ex,
                     fp64_frac=ex / fp64_peak, fp64_frac_of_nominal=ex / fp64_nominal,
                     # issue-slot view: FP64-pipe instructions per second over the probe's DFMA rate (one slot each)
                     fp64_pipe_frac=EXECUTED_PER_LEG["fp64_pipe_instr"][key] * n_legs / sec / (fp64_peak * 1e12 / 2.0),
                     fp64_pipe_pct_ncu=EXECUTED_PER_LEG["fp64_pipe_pct_ncu"][key])
        return k

    kf_fwd = kernel_roof("kf_forward_kernel", "kf_forward_kernel", fwd, fwd_bytes)
    kf_rts = kernel_roof("kf_mbf_kernel" if bf else "kf_rts_kernel", "kf_rts_kernel", rts, rts_bytes) if smooth else None
    dom = kf_fwd if (kf_rts is None or fwd >= rts) else kf_rts
    dkey = "kf_forward_kernel" if dom is kf_fwd else "kf_rts_kernel"
    # the dominant kernel's own bound: whichever roof it is nearer to (FP64 issue slots or HBM bytes)
    # (decided on the two fractions that are printed: executed flop / DFMA probe against algorithmic bytes / measured HBM)
    if exe_ok and dom["fp64_frac"] >= dom["hbm_frac"]:
        roofline = dict(bound="alu", achieved=dom["executed_tflops"], peak=fp64_peak, unit="TFLOP/s",
                        frac=dom["fp64_frac"], traffic=None, kernel=dom["kernel"],
                        what="EXECUTED FP64 flop (ncu opcode counts: " + EXECUTED_PER_LEG["source"] + ") / CUDA-event time, over the "
                             "DFMA-chain probe of the same run",
                        peak_source="kf_probe_fp64_tflops this run (8 independent DFMA chains per thread, all SMs)",
                        peak_nominal=fp64_nominal,
                        peak_nominal_source=f"148 SMs x {FP64_LANES_PER_SM} FP64 FMA lanes x 2 x {peaks['sm_max_mhz']:.0f} MHz (DESIGN.md)",
                        frac_of_nominal=dom["fp64_frac_of_nominal"], fp64_pipe_frac=dom["fp64_pipe_frac"],
                        fp64_pipe_pct_ncu=dom["fp64_pipe_pct_ncu"], hbm_frac=dom["hbm_frac"],
                        algorithmic=dict(flop_per_leg=alg[dkey], tflops=dom["algorithmic_tflops"],
                                         source=ALGORITHMIC_FLOP_PER_LEG["source"],
                                         note="the method's hand count; not comparable with a measured peak (the kernels "
                                              "execute fewer flop than the method states)"))
    else:
        roofline = dict(bound="hbm", achieved=dom["hbm_gbs"], peak=hbm_peak, unit="GB/s", frac=dom["hbm_frac"],
                        traffic=None, kernel=dom["kernel"], peak_source=f"MEASURED_PEAKS.json ({peaks['source']})",
                        what="ALGORITHMIC bytes (records + hits + per-track in/out of this launch) / CUDA-event time",
                        fp64_frac=dom.get("fp64_frac"), fp64_frac_of_nominal=dom.get("fp64_frac_of_nominal"),
                        fp64_pipe_frac=dom.get("fp64_pipe_frac"), fp64_pipe_pct_ncu=dom.get("fp64_pipe_pct_ncu"),
                        fp64_probe_tflops=fp64_peak, fp64_nominal_tflops=fp64_nominal)
    # the kernel sits near the ridge of its two roofs: both fractions as peers, whichever one `bound` names
    roofline["fracs"] = dict(hbm=dom["hbm_frac"], fp64=dom.get("fp64_frac"), fp64_pipe_ncu_pct=dom.get("fp64_pipe_pct_ncu"))
    roofline["ridge"] = bool(dom.get("fp64_frac") is not None and abs(dom["fp64_frac"] - dom["hbm_frac"]) < 0.2)
    roofline["executed_counts"] = "from " + EXECUTED_PER_LEG["source"] if exe_ok else "null: " + "; ".join(why_not)
    if exe_ok:  # the capture is of this workload, these kernels and these sources; else null
        roofline["traffic"] = NCU_TRAFFIC["bytes_per_leg"][dkey] * n_legs
        roofline["traffic_unit"] = "bytes per launch (ncu dram read+write per leg x legs of this launch)"
        roofline["traffic_source"] = NCU_TRAFFIC["source"]
    roofline["algorithmic_bytes"] = fwd_bytes if dom is kf_fwd else rts_bytes
    roofline["ms_per_launch"] = dom["ms"]
    roofline["share_of_step"] = dom["ms"] / ms_step
    # whole step against its two floors (kernels run back to back): executed flop / probe, algorithmic bytes / HBM peak
    if exe_ok:
        roofline["step_floors_ms"] = dict(
            fp64=(EXECUTED_PER_LEG["flop"]["kf_forward_kernel"] + EXECUTED_PER_LEG["flop"]["kf_rts_kernel"]) * n_legs
                 / (fp64_peak * 1e12) * 1e3,
            hbm=(fwd_bytes + rts_bytes) / (hbm_peak * 1e9) * 1e3, measured=ms_step)

    cpu = None if args.no_cpu_baseline else cpu_baseline(wl)

    # ---- context: the paper's own arithmetic on the same batch, clearly apart from the headline ----
    alt = None
    if not mixed and not bf and world == 1 and not args.field_gradient and not args.no_alt_precision:
        try:
            acall = kf.FitCall(db, out=out, variant=variant, precision=1)
            for _ in range(3):
                acall.run()
            torch.cuda.synchronize()
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record()
            for _ in range(args.steps):
                acall.run()
            a1.record()
            torch.cuda.synchronize()
            ams = a0.elapsed_time(a1) / args.steps
            alt = dict(precision="mixed", dtype="f32 (6x6 solve f64)", ms_per_step=ams, value=N / (ams * 1e-3), unit=UNIT,
                       note="kf_options.precision = MIXED on the same resident batch (float operands and records, the "
                            "smoother's 6x6 solve in double: the paper's operating point); context, not the metric")
            del acall
        except kf.KfError as e:   # a combination MIXED does not support
            alt = dict(precision="mixed", unavailable=str(e))

    line = dict(
        metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
        ms_per_step=ms_step, higher_is_better=True, scaling="weak", vs_baseline=None,
        dtype="f32 (6x6 solve f64)" if mixed else "f64",
        data="synthetic",
        config=dict(workload=W.WORKLOAD_NAMES[args.config], tracks=N, hits=M, legs=n_legs,
                    layers=hb.n_surfaces - 1, field=fkind, smooth=int(smooth),
                    material=int(hb.options.get("material", 0)),
                    l2="inputs larger than L2 (RTS workspace %.1f GB per step)" % (n_legs * rec_b / 1e9),
                    parallelism="replicas only" if world > 1 else "1 GPU", variant=args.variant, smoother=args.smoother,
                    precision=args.precision, field_gradient=int(args.field_gradient), field_stage=(fkind == "grid3" and args.field_stage),
                    extra_untimed_warmup_steps=extra_warmup, build_defines=kbuild.built_defines(), perigee=bool(args.perigee),
                    tracks_not_fitted=bad),
        clocks=clocks, e2e=e2e, gpu_launches=launches, roofline=roofline,
        kernels=[k for k in (kf_fwd, kf_rts) if k], fp64_probe_tflops=fp64_probe, cpu_baseline=cpu,
        step_stats=step_stats, alt_precision=alt)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
