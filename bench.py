#!/usr/bin/env python
"""bench.py -- channel-terms/s of the e-ph collision-integral hot path on B200 (BASELINE.json metric).

One "step" = one pass of the whole hot path over one workload.  The headline line is
quoted on the largest single-GPU config (gaas, BASELINE.json configs[2], 1.9e8 channels); the Si-like transport
config (configs[1]; configs[4] is the same channel set), the large-cell config and the tiny config are timed in
shorter runs and reported under `per_config`:
    1 collision evaluation + 1 transport_setup + 20 transport iterations (3 Cartesian components)
    + 1 RK4 rt-BTE step (4 collision evaluations with fused axpy) + the conservation scalar
  = 26 channel-loop evaluations; channel-terms per step = 26 * N_ch (N_ch = unordered active channels).

`value`     device-resident: inputs in HBM before the timed region, CUDA events on the launching stream.
`e2e`       the same step through the *_host entry points of the C ABI: pinned host buffers, H2D/D2H inside.
`roofline`  for the COLLISION call (the kernel north_star's target names): algorithmic bytes per launch (DESIGN.md
            "Roofline") / mean launch duration measured here with CUDA events, vs MEASURED_PEAKS.json; `kernels`
            holds the same figures for every call; `collision_channel_terms_per_s` is the collision call alone.
`cpu_baseline`  the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload: serial, and
            (`all_cores`) the paper's Baseline-CPU shape, OpenMP over the channel list with atomic updates.

--impl reference  times the oracle instead (rank 0 only).  N > 1: ONE problem, k-sharded over the ranks with an
all-gather of the owned slices after every evaluation ("strong"); --replicas runs one
independent problem per GPU instead ("weak", no collective).
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

N_TRANSPORT_ITERS = 20
EVALS_PER_STEP = 1 + 1 + N_TRANSPORT_ITERS + 4
METRIC = "collision-integral channel-terms/s (fp64)"
UNIT = "channel-terms/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="gaas",
                    help="workload: gaas (default: the largest single-GPU config, BASELINE configs[2]) | si | bigcell | tiny")
    ap.add_argument("--grid", type=int, default=0, help="override the grid edge (smaller copies for quick runs)")
    ap.add_argument("--pair-prob", type=float, default=0.0)
    ap.add_argument("--variant", type=int, default=-1,
                    help="-1: automatic (library default), 0: gather, 1: tiles, 2: stream, 3: resident tiles")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the short runs of the other configs")
    ap.add_argument("--sharded", action="store_true", help="use the k-sharded driver even with one rank")
    ap.add_argument("--replicas", action="store_true",
                    help="N > 1: independent replicas (weak scaling, no collective) instead of the k-sharded problem")
    return ap.parse_args()


def make_workload(args, seed_offset=0):
    from ephc_inputs import make_problem
    kw = {}
    if args.grid:
        kw["grid"] = (args.grid,) * 3
    if args.pair_prob:
        kw["pair_prob"] = args.pair_prob
    if seed_offset:
        kw["seed"] = 20251103 + 100 * seed_offset + 1
    return make_problem(args.config, **kw)


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            c = [x.strip() for x in r.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for n, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------------
def oracle_step(L, p, n_iters, n_rt):
    """The same step on the CPU oracle (bounded: n_iters transport iterations, n_rt RK4 steps)."""
    L.collision(p.f, p.N)
    G = L.transport_setup(p.f0, p.N)
    tau = np.where(G > 0, 1.0 / np.where(G > 0, G, 1.0), 0.0)
    F = tau[None, :] * p.v
    for _ in range(n_iters):
        F = L.transport_iter(p.f0, p.N, F, p.v, tau)
    if n_rt:
        L.rt_step(p.f, p.N, 1.0, n_rt)
    return 1 + 1 + n_iters + 4 * n_rt


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    p = make_workload(args)
    L = oracle.OracleList(p)
    # bounded sample per step, sized so that the run ends within minutes: collision + setup + n_iters transport
    # iterations + n_rt RK4 steps; the rate is per evaluation, so the sample stands for the whole step
    n_iters, n_rt = (2, 1) if L.nch < 5e7 else (1, 0)
    for _ in range(max(args.warmup, 0)):
        oracle_step(L, p, 0, 0) if L.nch < 5e7 else L.collision(p.f, p.N)
    t0 = time.perf_counter()
    evals = 0
    for _ in range(args.steps):
        evals += oracle_step(L, p, n_iters, n_rt)
    dt = time.perf_counter() - t0
    val = L.nch * evals / dt
    sample = (f"per step: 1 collision + 1 transport_setup + {n_iters} transport iterations + {n_rt} RK4 steps "
              f"({evals // max(args.steps, 1)} of the {EVALS_PER_STEP} evaluations of a full step; the rate per evaluation is "
              f"extrapolated to the step), full channel set, serial C")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(args, p, L.nch),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def reduce_over_ranks(dist, dev, ms_total, nch):
    """Replicas: the job's time is the MAX over ranks, its work the SUM of the ranks' channels."""
    if dist is None:
        return float(ms_total), float(nch)
    import torch
    t = torch.tensor([ms_total], device=dev, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    tot = torch.tensor([float(nch)], device=dev, dtype=torch.float64)
    dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    return float(t.item()), float(tot.item())


def workload_config(args, p, nch):
    return {"workload": f"{p.name}: {p.grid[0]}x{p.grid[1]}x{p.grid[2]} k-grid, window [{p.emin},{p.emax}] eV, "
                        f"{p.nk} active k, {p.nb} bands, {p.nnu} modes, sigma={p.sigma} eV",
            "n_channels": int(nch), "n_states": int(p.ns), "n_pairs_candidate": int(p.npair),
            "step": f"1 collision + 1 transport_setup + {N_TRANSPORT_ITERS} transport_iter (3 components) + 1 RK4 "
                    f"rt_step (4 evaluations) + sum f = {EVALS_PER_STEP} channel-loop evaluations",
            "seed": int(p.seed)}


def measure(args, ephc, torch, config_name, steps, warmup, rank, local, dist, with_e2e, with_cpu, sampler=None, with_paper=True):
    """Builds one workload and times `steps` steps of the whole hot path on it.  Returns a dict of results."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    dev = torch.device("cuda", local)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    a2 = argparse.Namespace(**vars(args))
    a2.config = config_name
    t0 = time.perf_counter()
    p = make_workload(a2, seed_offset=rank)       # replicas: an independent problem per rank
    t_gen = time.perf_counter() - t0
    t0 = time.perf_counter()
    h = ephc.build_channels(p, flags=ephc.TRANSPORT_COLLAPSE)   # + the mode-collapsed row store, timed separately below
    t_build = time.perf_counter() - t0
    if args.variant >= 0:
        h.set_variant(args.variant)
    variant, tvariant = h.get_variant(), h.get_transport_variant()
    q = h.query()
    nch, ns = q["nch"], p.ns

    def d(x):
        return torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64).reshape(-1), device=dev)

    f, f0, N, v = d(p.f), d(p.f0), d(p.N), d(p.v)
    I = torch.empty(ns, device=dev, dtype=torch.float64)
    G = torch.empty(ns, device=dev, dtype=torch.float64)
    tau = torch.empty(ns, device=dev, dtype=torch.float64)
    Fa = torch.empty(3 * ns, device=dev, dtype=torch.float64)
    Fb = torch.empty(3 * ns, device=dev, dtype=torch.float64)
    frt = f.clone()
    sumf = torch.zeros(2, device=dev, dtype=torch.float64)
    stream = torch.cuda.current_stream()

    def step(ev=None):
        """ev: list collecting the events that bracket the phases."""
        def mark():
            e = torch.cuda.Event(enable_timing=True)
            e.record(stream)
            return e
        e0 = mark() if ev is not None else None
        h.collision(f, N, I, stream)
        e1 = mark() if ev is not None else None
        h.transport_setup(f0, N, G, stream)
        e2 = mark() if ev is not None else None
        h.transport_start(G, v, tau, Fa, stream)
        e3 = mark() if ev is not None else None
        h.transport_iters(Fa, v, tau, Fb, N_TRANSPORT_ITERS, stream)   # 20 chained iterations (one public call)
        e4 = mark() if ev is not None else None
        h.rt_step(frt, N, 1.0, 1, sumf, stream)
        e5 = mark() if ev is not None else None
        if ev is not None:
            ev.append((e0, e1, e2, e3, e4, e5))

    for _ in range(max(warmup, 0)):
        step()
    barrier()
    if sampler is not None:
        sampler.start()
    l0 = h.launch_count()
    ev = []
    start, stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    start.record(stream)
    for _ in range(steps):
        step(ev)
    stop.record(stream)
    barrier()
    clocks = sampler.stop() if sampler is not None else None
    launches = h.launch_count() - l0
    ms_total, nch_all = reduce_over_ranks(dist, dev, start.elapsed_time(stop), nch)
    value = nch_all * EVALS_PER_STEP * steps / (ms_total * 1e-3)

    # per-phase device times (this rank)
    ph = np.array([[e[i].elapsed_time(e[i + 1]) for i in range(5)] for e in ev]) if ev else np.zeros((1, 5))
    ms_coll, ms_setup, ms_tau, ms_iter, ms_rt = ph.mean(axis=0)
    peak, peak_src = peaks()
    kern = {}
    traffic = load_traffic(p.name)

    def roof(call, kernels, ms_launch, alg_bytes, share):
        gbs = alg_bytes / (ms_launch * 1e-3) / 1e9 if ms_launch > 0 else 0.0
        tr = traffic.get(call)
        kern[f"{call} ({kernels})"] = {
            "bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
            "traffic": tr["bytes"] if tr else None, "traffic_source": tr["source"] if tr else None,
            "frac_of_nominal_8TBs": gbs / 8000.0,
            "frac_dram_traffic": (tr["bytes"] / (ms_launch * 1e-3) / 1e9 / peak) if (tr and ms_launch > 0) else None,
            "alg_bytes_per_launch": int(alg_bytes), "us_per_launch": 1e3 * ms_launch, "share_of_step": share,
            "channel_terms_per_s": nch / (ms_launch * 1e-3) if ms_launch > 0 else 0.0}

    ms_step = ms_total / max(steps, 1)
    cname = {0: "gather_kernel<0>", 1: "tile_kernel<0> + finish_kernel<0>", 2: "stream_kernel + finish_kernel<0>",
             3: "res_compact_kernel + res_kernel + finish_kernel<0>"}[variant]
    rname = {0: "gather_kernel<1>", 1: "tile_kernel<0> + finish_kernel<1>", 2: "stream_kernel + finish_kernel<1>",
             3: "res_kernel + finish_kernel<1>, which also writes the next stage's compact f"}[variant]
    sname, iname = "row_compact1_kernel + row_setup_kernel", "row_iter_kernel (+ one row_compact_kernel per 20 chained iterations)"
    if os.environ.get("EPHC_NO_ROWS"):
        sname, iname = "gather_kernel<2>", "gather_kernel<3>"
    if tvariant == 1:
        sname, iname = "tile_kernel<2> + finish_kernel<2>", "tile_kernel<3> + finish_kernel<3>"
    roof("collision", cname, ms_coll, q["alg_bytes_collision"], ms_coll / ms_step)
    # the collision bytes plus the 16 bytes of weights per channel that the setup produces
    roof("transport_setup", sname, ms_setup, q["alg_bytes_collision"] + 16 * nch, ms_setup / ms_step)
    roof("transport_iter", iname, ms_iter / N_TRANSPORT_ITERS, q["alg_bytes_transport"], ms_iter / ms_step)
    # an RK stage moves the collision bytes plus the fused axpy vectors (f0, ksum r/w, ynext): 32 B per state
    roof("rk4 stage", rname, ms_rt / 4, q["alg_bytes_collision"] + 32 * ns, ms_rt / ms_step)
    coll_key = next(k for k in kern if k.startswith("collision"))
    roofline = dict(kern[coll_key], kernel=coll_key, peak_source=peak_src)
    # A/B on the same GPU: the paper's own layout and two-step algorithm as variant 4
    if with_paper:
        h.set_variant(4)
        for _ in range(3):
            h.collision(f, N, I, stream)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(10):
            h.collision(f, N, I, stream)
        e1.record(stream)
        torch.cuda.synchronize()
        ms_paper = e0.elapsed_time(e1) / 10
        roof("paper-layout collision", "paper_step2_kernel + paper_step3_kernel", ms_paper, q["alg_bytes_collision"], 0.0)
        kern[next(k for k in kern if k.startswith("paper-layout"))]["note"] = (
            "not part of the step: PAPER.md:84-102 as two plain kernels on the same problem, for comparison; its own layout moves "
            "about %.0f B per channel" % ((24 * q["nw"] + 8 * q["nw"] * 2 + 8 * q["nw"] * 2) / max(nch, 1)))
        h.set_variant(args.variant)

    # the mode-collapsed transport specialisation (SURVEY.md 8(d) honesty note): 20 chained iterations on one weight per
    # (destination, partner) state pair.  Fewer bytes per claimed channel-term: reported here, never part of `value`.
    if with_paper and h.collapsed_entries() > 0 and tvariant == 0 and not os.environ.get("EPHC_NO_ROWS"):
        ec0, ec1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ec0.record(stream)
        h.transport_collapse(stream)          # sums the weights of the last transport_setup per state pair; switches over
        ec1.record(stream)
        for _ in range(2):
            h.transport_iters(Fa, v, tau, Fb, N_TRANSPORT_ITERS, stream)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(3):
            h.transport_iters(Fa, v, tau, Fb, N_TRANSPORT_ITERS, stream)
        e1.record(stream)
        torch.cuda.synchronize()
        h.set_transport_collapsed(False)
        ms_c = e0.elapsed_time(e1) / (3 * N_TRANSPORT_ITERS)
        nc = h.collapsed_entries()
        bytes_c = 10 * nc + (3 * 8 * 3 + 8) * ns
        kern["transport_iter, mode-collapsed specialisation (row_iter_kernel on one weight per state pair)"] = {
            "bound": "hbm", "achieved": bytes_c / (ms_c * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
            "frac": bytes_c / (ms_c * 1e-3) / 1e9 / peak, "traffic": None, "alg_bytes_per_launch": int(bytes_c),
            "us_per_launch": 1e3 * ms_c, "share_of_step": 0.0, "channel_terms_per_s": nch / (ms_c * 1e-3),
            "state_pairs": int(nc), "ordered_terms": int(q["gather_entries"]),
            "note": "not part of the step or of `value`: a specialisation that moves %.1f B per channel-term instead of %.1f; "
                    "`achieved` counts ITS bytes (10 B per state pair + the vectors), `channel_terms_per_s` the channel terms it "
                    "stands for; general path: %.1f us per iteration; summing the weights once per setup (row_collapse_kernel): %.1f us"
                    % (bytes_c / max(nch, 1), q["alg_bytes_transport"] / max(nch, 1), 1e3 * ms_iter / N_TRANSPORT_ITERS,
                       1e3 * ec0.elapsed_time(ec1))}

    # ---- end to end: the same step through host buffers ------------------------------------------------
    e2e = None
    if with_e2e:
        pin = lambda x: torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64).reshape(-1)).pin_memory()
        hf, hf0, hN, hv = pin(p.f), pin(p.f0), pin(p.N), pin(p.v)
        hI, hF, hG = pin(np.zeros(ns)), pin(np.zeros(3 * ns)), pin(np.zeros(ns))
        hfrt, hs = pin(p.f), pin(np.zeros(2))

        def step_host():
            h.collision_host(hf, hN, hI)
            h.transport_solve_host(hf0, hN, hv, N_TRANSPORT_ITERS, hF, hG)
            h.rt_step_host(hfrt, hN, 1.0, 1, hs)
        h2d = 8 * (ns + p.nq * p.nnu) + 8 * (ns + p.nq * p.nnu + 3 * ns) + 8 * (ns + p.nq * p.nnu)
        d2h = 8 * ns + 8 * (3 * ns + ns) + 8 * (ns + 2)
        for _ in range(max(warmup, 0)):
            step_host()
        barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            step_host()
        barrier()
        dt = time.perf_counter() - t0
        if dist is not None:
            t = torch.tensor([dt], device=dev, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": nch_all * EVALS_PER_STEP * steps / dt, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "ms_per_step": 1e3 * dt / max(steps, 1)}

    # ---- CPU oracle on a bounded sample (rank 0, N = 1 only): serial, and the paper's Baseline-CPU shape on all cores --
    cpu = None
    if with_cpu:
        import oracle
        L = oracle.OracleList(p)
        assert L.nch == nch, "oracle and library disagree on the channel count"
        n_it = 4 if nch < 5e7 else 1
        t0 = time.perf_counter()
        evals = oracle_step(L, p, n_it, 1)
        dt = time.perf_counter() - t0
        ncore = oracle.threads()
        L.collision(p.f, p.N, omp=True)
        t1 = time.perf_counter()
        nomp = 3
        for _ in range(nomp):
            L.collision(p.f, p.N, omp=True)
        dto = time.perf_counter() - t1
        cpu = {"value": L.nch * evals / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"one pass: 1 collision + 1 transport_setup + {n_it} transport iterations + 1 RK4 step = {evals} of the "
                         f"{EVALS_PER_STEP} evaluations of a step, full channel set ({dt:.1f} s, serial C, gcc -O2)",
               "all_cores": {"value": L.nch * nomp / dto, "unit": UNIT, "cores": int(ncore), "kind": "oracle",
                             "sample": f"{nomp} collision evaluations, OpenMP over the channel list with atomic updates "
                                       f"(the paper's Baseline-CPU shape, PAPER.md:74), {dto:.1f} s"},
               "host_cores_available": os.cpu_count()}
        del L

    cfg = workload_config(a2, p, nch)
    sb = {0: q["store_bytes_gather"], 1: q["store_bytes_scatter"], 2: q["store_bytes_scatter"], 3: q["store_bytes_scatter"]}[variant]
    if variant != 0 and tvariant == 0:
        sb += q["store_bytes_gather"]
    names = {0: "gather", 1: "tiles", 2: "stream", 3: "resident tiles"}
    tname = names[tvariant] if (tvariant == 1 or os.environ.get("EPHC_NO_ROWS")) else "rows"
    coll_mb = (q["store_bytes_scatter"] if variant else q["store_bytes_gather"]) / 1e6
    l2 = ("no flush: every collision evaluation streams its %.0f MB store, larger than the 126 MB L2" % coll_mb
          if coll_mb > 126 else "no flush: the %.0f MB collision store FITS the 126 MB L2 (L2-resident after warm-up; the roofline fraction is not an HBM figure)" % coll_mb)
    cfg.update({"variant": f"collision/rt: {names[variant]}, transport: {tname}", "l2": l2,
                "parallelism": "1 GPU" if world == 1 else f"{world} independent replicas (one problem per GPU, no data-path collective)",
                "generate_s": t_gen, "build_channels_s": t_build, "store_bytes": sb + q["store_bytes_transport"],
                "store_bytes_per_channel": (sb + q["store_bytes_transport"]) / max(nch, 1)})
    h.close()
    # the kernel with the largest share of the step (the transport iteration), beside the collision call in `roofline`
    dom_key = max((k for k in kern if kern[k]["share_of_step"] > 0), key=lambda k: kern[k]["share_of_step"])
    return {"value": value, "ms_per_step": ms_step, "config": cfg, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
            "roofline": roofline, "roofline_dominant": dict(kern[dom_key], kernel=dom_key, peak_source=peak_src), "kernels": kern,
            "cpu_baseline": cpu,
            "collision_channel_terms_per_s": nch_all / (ms_coll * 1e-3) if ms_coll > 0 else 0.0}


def measure_sharded(args, ephc, torch, rank, local, dist):
    """N > 1: ONE problem, k-sharded over the ranks: every rank owns a range
    of destination k points, computes its states and exchanges the owned slices with an NCCL all-gather after every
    evaluation (collision, Gamma, every transport iteration, every RK stage).  Strong scaling: the total work is fixed."""
    from paper_2511_03683_b200.sharded import ShardedSolver
    world = dist.get_world_size()
    dev = torch.device("cuda", local)

    def barrier():
        dist.barrier()
        torch.cuda.synchronize()

    t0 = time.perf_counter()
    p = make_workload(args)                       # the same problem on every rank
    t_gen = time.perf_counter() - t0
    t0 = time.perf_counter()
    S = ShardedSolver(p, dist, dev)
    t_build = time.perf_counter() - t0
    q = S.h.query()
    nch, ns = q["nch"], p.ns

    def d(x):
        return torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64).reshape(-1), device=dev)

    pin = lambda x: torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64).reshape(-1)).pin_memory()
    hf, hf0, hN, hv = pin(p.f), pin(p.f0), pin(p.N), pin(p.v)
    f, f0, N, v = d(p.f), d(p.f0), d(p.N), d(p.v)
    I, G, tau = (torch.empty(ns, device=dev, dtype=torch.float64) for _ in range(3))
    Fa, Fb = (torch.empty(3 * ns, device=dev, dtype=torch.float64) for _ in range(2))
    frt = f.clone()
    hI, hF, hfrt = pin(np.zeros(ns)), pin(np.zeros(3 * ns)), pin(np.zeros(ns))
    stream = torch.cuda.current_stream()

    def step(host=False):
        if host:
            f.copy_(hf, non_blocking=True); f0.copy_(hf0, non_blocking=True)
            N.copy_(hN, non_blocking=True); v.copy_(hv, non_blocking=True); frt.copy_(hf, non_blocking=True)
        S.collision(f, N, I, stream)
        F = S.transport_solve(f0, N, v, N_TRANSPORT_ITERS, G, tau, Fa, Fb, stream)
        S.rt_step(frt, N, 1.0, 1, stream)
        if host:
            hI.copy_(I, non_blocking=True); hF.copy_(F, non_blocking=True); hfrt.copy_(frt, non_blocking=True)
            torch.cuda.synchronize()

    def timed(host):
        for _ in range(max(args.warmup, 0)):
            step(host)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = S.h.launch_count()
        e0.record(stream)
        for _ in range(args.steps):
            step(host)
        e1.record(stream)
        barrier()
        t = torch.tensor([e0.elapsed_time(e1)], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item()), S.h.launch_count() - l0

    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    ms_total, launches = timed(False)
    clocks = sampler.stop() if sampler else None
    ms_e2e, _ = timed(True) if not args.no_e2e else (None, 0)
    lo, hi = S.h.owned_states()
    own = [None] * world
    dist.all_gather_object(own, [lo, hi, int(S.h.query()["gather_entries"])])
    # the collision call alone (every rank: it ends in a collective)
    ec = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    for _ in range(3):
        S.collision(f, N, I, stream)
    barrier()
    ec[0].record(stream)
    for _ in range(10):
        S.collision(f, N, I, stream)
    ec[1].record(stream)
    barrier()
    ms_c = ec[0].elapsed_time(ec[1]) / 10
    if rank != 0:
        return None
    exchanges = 1 + 1 + N_TRANSPORT_ITERS * 3 + 4
    cfg = workload_config(args, p, nch)
    cfg.update({"variant": "collision/rt: gather (destination-sorted, two-sided), transport: rows",
                "parallelism": f"k-sharded over {world} GPUs: contiguous ranges of destination k balanced by half-pair count; "
                               f"{exchanges} all-gathers of the owned slices per step (NCCL), <= {8 * ns} bytes each",
                "owned_states_and_ordered_entries_per_rank": own, "generate_s": t_gen, "build_channels_s": t_build,
                "l2": "no flush: every rank streams its share of the two-sided store in every evaluation"})
    val = nch * EVALS_PER_STEP * args.steps / (ms_total * 1e-3)
    # roofline of the collision call on this rank's share (gather_kernel<0> + the all-gather of the owned slice): the
    # algorithmic bytes of the whole problem times the share of the ordered terms rank 0 owns
    share0 = own[0][2] / max(sum(o[2] for o in own), 1)
    peak, peak_src = peaks()
    gbs = q["alg_bytes_collision"] * share0 / (ms_c * 1e-3) / 1e9
    roofline = {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "traffic": None,
                "kernel": "collision on rank 0's share (gather_kernel<0> + NCCL all-gather of the owned slice)",
                "alg_bytes_per_launch": int(q["alg_bytes_collision"] * share0), "us_per_launch": 1e3 * ms_c,
                "share_of_ordered_terms": share0, "peak_source": peak_src}
    e2e = None
    if ms_e2e is not None:
        e2e = {"value": nch * EVALS_PER_STEP * args.steps / (ms_e2e * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": int(8 * (3 * ns + p.nq * p.nnu + 3 * ns)), "d2h_bytes_per_step": int(8 * 5 * ns),
               "ms_per_step": ms_e2e / max(args.steps, 1)}
    return {"metric": METRIC, "value": val, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total / max(args.steps, 1), "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": cfg, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
            "roofline": roofline, "cpu_baseline": None}


def load_traffic(config_name):
    """DRAM bytes per launch from the committed `ncu --set full` captures (cold caches: ncu flushes them per kernel)."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    out = {}
    if os.path.exists(path):
        import csv
        with open(path, newline="") as fh:
            for row in csv.DictReader(fh):
                if row.get("config") == config_name:
                    out[row["call"]] = {"bytes": int(row["dram_bytes_per_launch"]),
                                        "source": f"ncu --set full, cold caches, build {row.get('build', '?')} ({row.get('capture', '')})"}
    return out


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import paper_2511_03683_b200 as ephc

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    if args.sharded and world == 1:            # the sharded driver with a single rank (checks the code path on one GPU)
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29533")
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", local))
    if (world > 1 and not args.replicas) or args.sharded:
        out = measure_sharded(args, ephc, torch, rank, local, dist)
        if rank == 0:
            print(json.dumps(out))
        dist.destroy_process_group()
        return
    sampler = ClockSampler(local) if rank == 0 else None
    main_res = measure(args, ephc, torch, args.config, args.steps, args.warmup, rank, local, dist,
                       with_e2e=not args.no_e2e, with_cpu=(rank == 0 and world == 1 and not args.no_cpu_baseline), sampler=sampler)
    # the other BASELINE.json configs, shorter runs, device-resident only (parity is the tests' job)
    per_config = {}
    if world == 1 and not args.no_per_config and not args.grid:
        for name in ("si", "bigcell", "tiny"):
            if name == args.config:
                continue
            r = measure(args, ephc, torch, name, max(3, args.steps // 2), 3, rank, local, None, with_e2e=False, with_cpu=False)
            per_config[name] = {k: r[k] for k in ("value", "ms_per_step", "collision_channel_terms_per_s", "config", "kernels")}
            per_config[name]["unit"] = UNIT
    if rank == 0:
        out = {"metric": METRIC, "value": main_res["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
               "warmup": args.warmup, "ms_per_step": main_res["ms_per_step"], "higher_is_better": True, "scaling": "weak",
               "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": main_res["config"], "e2e": main_res["e2e"],
               "gpu_launches": main_res["gpu_launches"], "clocks": main_res["clocks"], "roofline": main_res["roofline"],
               "roofline_dominant": main_res["roofline_dominant"],
               "collision_channel_terms_per_s": main_res["collision_channel_terms_per_s"],
               "kernels": main_res["kernels"], "cpu_baseline": main_res["cpu_baseline"], "per_config": per_config}
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
