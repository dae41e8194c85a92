"""bench.py -- events/s of the whole hot path (Philox+RAMBO+cuts -> helicity- and colour-summed |M|^2) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C5] [--precision fp64] [--impl ours|reference]

One "step" = one pass of steps a1-a8 over one batch of E synthetic events: heget_sample_momenta then
heget_eval_me2 on device-resident buffers.  BASELINE.json's metric is "per process" and quotes no single config, so the
headline line sits on the largest single-GPU config -- C5, u u~ -> g g g g g, 2^18 events, sqrt(s_hat) = 2 TeV, FP64 --
and the same JSON line carries `per_config`: every config C1-C5 in FP64 and FP32 (a few steps each, same timing rules).
Prints ONE JSON line (rank 0).  N > 1: one process per GPU under torchrun (`--gpus N` without a launcher starts the ranks
itself), every rank takes E events of its own global range (weak scaling, no collective on the data path).
`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
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

CONFIGS = {   # BASELINE.json configs / SURVEY.md 8 table: process, sqrt(s_hat) [GeV], events, Philox seed
    "C1": ("u u~ > g g", 500.0, 1 << 14, 0),
    "C2": ("g g > g g g", 1000.0, 1 << 20, 1),
    "C3": ("u u > u u g g", 1000.0, 1 << 20, 2),
    "C4": ("g g > g g g g", 1500.0, 1 << 20, 3),
    "C5": ("u u~ > g g g g g", 2000.0, 1 << 18, 4),
}
# events of the timed CPU-oracle sample (C4 the 4096-event validation subset; C5 512 of its 2048-event
# subset -- at ~30 events/s on 16 threads the whole subset would take over a minute, outside the 10-30 s the sample may cost)
ORACLE_SAMPLE = {"C1": 1 << 14, "C2": 1 << 15, "C3": 1 << 13, "C4": 1 << 12, "C5": 1 << 9}
# events per step of the reference arm (--impl reference runs warmup + steps of them: a few minutes in total)
REFERENCE_SAMPLE = {"C1": 1 << 14, "C2": 1 << 14, "C3": 1 << 12, "C4": 1 << 9, "C5": 1 << 7}
# executed floating-point operations per event of the |M|^2 kernels: ncu smsp__sass_thread_inst_executed_op_{d,f}{add,mul,fma}_pred_on.sum
# (FMA x 2) divided by the events of the profiled launch -- profiles/r2_opcounts.md.  Key: (config, precision, back end).
EXECUTED_FLOPS_PER_EVENT = {
    ("C1", "fp32", "straight"): 3580.0, ("C1", "fp64", "straight"): 4149.0,
    ("C2", "fp32", "straight"): 173643.0, ("C2", "fp64", "straight"): 175803.0,
    ("C3", "fp32", "straight"): 151170.0, ("C3", "fp64", "straight"): 152160.0,
    ("C4", "fp32", "table"): 1775299.0, ("C4", "fp64", "table"): 1776434.0,
    ("C5", "fp32", "table"): 6527332.0, ("C5", "fp64", "table"): 6485570.0,
}
METRIC = "helicity-summed |M|^2 events/sec per process on 1 B200; % of FP64/FP32 peak"
# dram__bytes_read.sum + dram__bytes_write.sum of the |M|^2 kernel, bytes per launch, from the committed `ncu --set full` captures
TRAFFIC = {("C2", "fp64"): 178.3e6, ("C2", "fp32"): 175.0e6,
           ("C5", "fp64"): 60.68e6, ("C5", "fp32"): 60.02e6, ("C4", "fp64"): 217.7e6, ("C4", "fp32"): 212.9e6}
TRAFFIC_NOTE = {("C2", "fp64"): "profiles/r1b_ncu_c2.md (algorithmic: 168 MB in + 8 MB out)", ("C2", "fp32"): "profiles/r1b_ncu_c2.md (algorithmic: 168 MB in + 4 MB out)",
                ("C5", "fp64"): "profiles/r2_ncu_table.md (algorithmic: 58.7 MB in + 2.1 MB out)",
                ("C5", "fp32"): "profiles/r2_ncu_table.md (algorithmic: 58.7 MB in + 1.0 MB out)",
                ("C4", "fp64"): "profiles/r2_ncu_table.md (algorithmic: 201.3 MB in + 8.4 MB out)",
                ("C4", "fp32"): "profiles/r2_ncu_table.md (algorithmic: 201.3 MB in + 4.2 MB out)",
                }
SM_COUNT, FP64_LANES, FP32_LANES = 148, 64, 128      # per SM; DESIGN.md "Roofline" derives the ALU peak from these


def peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


class ClockSampler:
    """nvidia-smi clocks line of /opt/skills/guides/B200_PROFILING.md, sampled during the timed region."""

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + q, "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, reasons, mx, pw = [], set(), None, []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx = float(r[1]); pw.append(float(r[2]))
                for k, nm in enumerate(names):
                    if r[3 + k].strip().lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        if sm:
            hi = [x for x in sm if x >= 0.5 * max(sm)]
            out = {"sm_mhz": statistics.median(hi), "sm_max_mhz": mx, "reasons": sorted(reasons), "samples": len(sm),
                   "power_w_max": max(pw) if pw else None}
        return out


def run_reference(a):
    """The CPU oracle, as it stands, on a bounded sample of the workload (host cores of this box)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as O
    name, sqrt_s, E, seed = CONFIGS[a.config]
    n = min(E, REFERENCE_SAMPLE[a.config])
    P = O.Process(name, 0.118)
    nf = P.n_ext - 2
    times = []
    for k in range(a.warmup + a.steps):
        t0 = time.perf_counter()
        mom, w, tr = O.sample_momenta(nf, sqrt_s, seed, n, first_event=k * n)
        me2 = P.me2(mom)
        dt = time.perf_counter() - t0
        if k >= a.warmup:
            times.append(dt)
    assert me2.min() > 0
    tot = sum(times)
    v = n * len(times) / tot
    cores = O.max_threads()
    sample = "%d of %d events per step (first events of the seed-%d stream), FP64, OpenMP over events" % (n, E, seed)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": "events/s", "n_gpus": a.gpus, "steps": a.steps, "warmup": a.warmup,
        "ms_per_step": 1e3 * tot / len(times), "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": "%s: %s, sqrt_s_hat=%g GeV, %d events/step" % (a.config, name, sqrt_s, E), "precision": "fp64"},
        "cpu_baseline": {"value": v, "unit": "events/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def measure(hg, torch, name, sqrt_s, E, seed, precision, steps, warmup, world, rank, first, barrier, max_over_ranks, kernel=None,
            lanes=0, use_graph=True, extras=True, colour_stage=None):
    """One (config, precision): K timed steps of sample + eval on device-resident buffers, the |M|^2 kernel alone, and the
    host-buffer end-to-end arm.  Returns a dict of raw numbers."""
    P = hg.Process(name, sqrt_s, precision=precision, kernel=kernel)
    if lanes:
        P.set_lanes(lanes)
    if colour_stage:
        P.set_colour_stage(colour_stage)
        extras = extras and colour_stage != "tensor"        # the tensor-core stage serves HEL_SUM only
    info = P.info
    ne = info.n_ext
    mom = torch.empty(ne, 4, E, dtype=torch.float64, device="cuda")
    wgt = torch.empty(E, dtype=torch.float64, device="cuda")
    me2 = torch.empty(E, dtype=P.dtype, device="cuda")
    need_flush = mom.numel() * 8 < (160 << 20)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda") if need_flush else None     # > 126 MB L2
    hg_count = [0]                        # kernels replayed from a CUDA graph (the library's own counter does not see replays)

    def step(k):
        P.sample_momenta(seed, E, first_event=first + k * world * E, mom=mom, weight=wgt)
        P.eval_me2(mom, out=me2)

    for k in range(warmup):
        step(k)
    barrier()
    # small batches (C1: 2^14 events, ~20 us of GPU work per kernel) are bound by the host's launch path: replay the step from
    # a CUDA graph.  The captured step re-samples the same event range each replay (first_event is baked into the graph).
    graph = None
    if E < (1 << 17) and use_graph:
        try:
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                step(0)
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=side):
                    step(0)
            torch.cuda.current_stream().wait_stream(side)
            torch.cuda.synchronize()
            graph = g
        except Exception as exc:       # capture not possible: plain launches
            graph = None
            sys.stderr.write("bench.py: CUDA graph capture failed (%s); timing plain launches\n" % exc)
            torch.cuda.synchronize()
    if graph is not None:
        def step(k):
            graph.replay()
            hg_count[0] += 2
        for k in range(warmup):
            step(k)
        barrier()
    clocks = ClockSampler(int(os.environ.get("LOCAL_RANK", "0"))) if rank == 0 else None
    c0 = hg.launch_count()
    hg_count[0] = 0
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * steps)]
    for k in range(steps):
        if need_flush:
            flush.fill_(k & 0xff)
        ev[2 * k].record()
        step(warmup + k)
        ev[2 * k + 1].record()
    barrier()
    launches = hg.launch_count() - c0 + hg_count[0]
    ms = sum(ev[2 * k].elapsed_time(ev[2 * k + 1]) for k in range(steps))
    ms = max_over_ranks(ms)
    clk = clocks.stop() if clocks else None
    assert bool(torch.isfinite(me2).all()) and float(me2.min()) > 0.0
    out = {"info": info, "E": E, "value": world * E * steps / (ms * 1e-3), "ms_per_step": ms / steps, "launches": int(launches), "clocks": clk,
           "graph": graph is not None, "need_flush": need_flush, "mom_mib": mom.numel() * 8 >> 20, "dtype": P.dtype}

    # ---- the dominant kernel alone (heget_eval_me2), for the roofline --------------------------------------------------
    kev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * steps)]
    for k in range(steps):
        if need_flush:
            flush.fill_(k & 0xff)
        kev[2 * k].record()
        P.eval_me2(mom, out=me2)
        kev[2 * k + 1].record()
    torch.cuda.synchronize()
    out["kernel_ms"] = sum(kev[2 * k].elapsed_time(kev[2 * k + 1]) for k in range(steps)) / steps
    sev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    sev[0].record()
    for k in range(steps):
        P.sample_momenta(seed, E, first_event=first, mom=mom, weight=wgt)
    sev[1].record()
    torch.cuda.synchronize()
    out["sampling_ms"] = sev[0].elapsed_time(sev[1]) / steps

    if extras:
        # what the paper itself timed: ONE Philox-drawn helicity configuration per event, for context
        P.eval_me2(mom, mode=hg.HEL_SAMPLE, seed=seed, first_event=first, out=me2)
        hev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        hev[0].record()
        for k in range(steps):
            P.eval_me2(mom, mode=hg.HEL_SAMPLE, seed=seed + k, first_event=first, out=me2)
        hev[1].record()
        torch.cuda.synchronize()
        out["hel_sample"] = E * steps / (hev[0].elapsed_time(hev[1]) * 1e-3)

    # ---- end to end through the C-ABI with HOST buffers ----------------------------------------------------------------
    h_mom = torch.empty(ne, 4, E, dtype=torch.float64).pin_memory()
    h_me2 = torch.empty(E, dtype=P.dtype).pin_memory()
    h_mom.copy_(mom)
    for k in range(2):
        P.run_host(seed, E, mom_in=h_mom, out=h_me2)
    barrier()
    t0 = time.perf_counter()
    for k in range(steps):
        P.run_host(seed, E, mom_in=h_mom, out=h_me2)
    barrier()
    e2e_s = max_over_ranks(time.perf_counter() - t0)
    out["e2e"] = world * E * steps / e2e_s
    out["h2d"] = int(h_mom.numel() * 8)
    out["d2h"] = int(h_me2.numel() * h_me2.element_size())
    P.close()
    del mom, wgt, me2, flush, h_mom, h_me2
    torch.cuda.empty_cache()
    return out


def roofline_of(m, precision, sm_max, cfg):
    """Counted and executed flop rates of the |M|^2 kernel against the nominal ALU peak."""
    info = m["info"]
    lanes = FP64_LANES if precision == "fp64" else FP32_LANES
    peak = SM_COUNT * lanes * 2 * sm_max * 1e6 / 1e12
    achieved = info.flops_per_event * m["E"] / (m["kernel_ms"] * 1e-3) / 1e12
    kname = "table" if info.kernel == 2 else "straight"
    ex = EXECUTED_FLOPS_PER_EVENT.get((cfg, precision, kname))
    executed = ex * m["E"] / (m["kernel_ms"] * 1e-3) / 1e12 if ex else None
    return {"achieved": achieved, "peak": peak, "frac": achieved / peak, "flops_per_event": info.flops_per_event,
            "executed_flops_per_event": ex, "executed": executed, "executed_frac": executed / peak if executed else None,
            "kernel_ms": m["kernel_ms"], "kernel": kname}


def cpu_baseline(name, sqrt_s, seed, E, cfg):
    """The oracle as it stands, timed on this box's host cores: all cores on the BASELINE.md section 3 sample, one core on 1/8 of it."""
    from oracle import oracle as O
    n = min(E, ORACLE_SAMPLE[cfg])
    Po = O.Process(name, 0.118)          # colour-matrix construction: outside the timed region
    ne = Po.n_ext
    t0 = time.perf_counter()
    m_o, _, _ = O.sample_momenta(ne - 2, sqrt_s, seed, n)
    Po.me2(m_o)
    dt = time.perf_counter() - t0
    cores = O.max_threads()
    n1 = max(1, n // 8)
    t0 = time.perf_counter()
    Po.me2(m_o[:, :, :n1].copy(), n_threads=1)
    dt1 = time.perf_counter() - t0
    Po.me2(m_o[:, :, :1].copy(), n_threads=cores)      # restore the thread count for later callers
    return {"value": n / dt, "unit": "events/s", "cores": cores, "kind": "oracle",
            "sample": "first %d of the %d seed-%d events, FP64, OpenMP static over events, %.1f s" % (n, E, seed, dt),
            "one_core": {"value": n1 / dt1, "unit": "events/s", "sample": "first %d events, 1 thread, %.1f s" % (n1, dt1)}}


def run_ours(a):
    import torch
    import torch.distributed as dist
    import paper_0909_5257_b200 as hg

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if a.gpus != world:
        if "WORLD_SIZE" in os.environ:
            raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d" % (a.gpus, world))
        # `python bench.py --gpus N` without a launcher: start the N ranks ourselves (one process per GPU, rendezvous on 127.0.0.1)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(a.gpus), "--master-addr", "127.0.0.1",
               "--master-port", str(29500 + os.getpid() % 2000), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    name, sqrt_s, E, seed = CONFIGS[a.config]
    if a.events:
        E = a.events                      # profiling aid only: not BASELINE.json's size, the workload string says so
    first = rank * E                      # weak scaling: rank r evaluates global events [rE, (r+1)E)
    m = measure(hg, torch, name, sqrt_s, E, seed, a.precision, a.steps, a.warmup, world, rank, first, barrier, max_over_ranks,
                kernel=a.kernel, lanes=a.lanes, use_graph=not a.no_graph, colour_stage=a.colour_stage)
    info = m["info"]
    pk = peaks()
    sm_max = float(pk.get("sm_max_mhz", 1965.0))
    roof = roofline_of(m, a.precision, sm_max, a.config)
    # measured FMA-chain peak of this GPU at the clock it holds under this kind of load
    prec = hg.FP64 if a.precision == "fp64" else hg.FP32
    nthr = SM_COUNT * 2048
    hg.fma_probe(prec, 1 << 12, nthr)
    torch.cuda.synchronize()
    pev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    pev[0].record()
    fl = hg.fma_probe(prec, 1 << 16, nthr)
    pev[1].record()
    torch.cuda.synchronize()
    probe = fl / (pev[0].elapsed_time(pev[1]) * 1e-3) / 1e12

    # ---- every BASELINE.json config in both precisions, a few steps each (same timing rules; rank 0's GPU at N = 1) ------------
    per_config = None
    if world == 1 and not a.no_sweep and not a.events:
        per_config = {}
        for cfg in sorted(CONFIGS):
            for prc in ("fp64", "fp32"):
                cn, cs, cE, cseed = CONFIGS[cfg]
                if cfg == a.config and prc == a.precision and a.kernel is None and not a.lanes and not a.colour_stage:
                    mm = m
                else:
                    mm = measure(hg, torch, cn, cs, cE, cseed, prc, a.sweep_steps, 3, 1, 0, 0, barrier, max_over_ranks, extras=False)
                r = roofline_of(mm, prc, sm_max, cfg)
                ci = mm["info"]
                per_config["%s/%s" % (cfg, prc)] = {
                    "process": cn, "events_per_step": cE, "events_per_s": mm["value"], "ms_per_step": mm["ms_per_step"], "kernel_ms": mm["kernel_ms"],
                    "kernel": r["kernel"], "frac": r["frac"], "executed_frac": r["executed_frac"], "counted_tflops": r["achieved"],
                    "flops_per_event": r["flops_per_event"], "executed_flops_per_event": r["executed_flops_per_event"],
                    "regs": ci.regs_per_thread, "local_bytes": ci.local_bytes_per_thread, "threads_per_block": ci.threads_per_block,
                    "j_in_tmem": ci.j_in_tmem, "warps_per_j": ci.warps_per_j, "e2e_events_per_s": mm["e2e"], "steps": a.steps if mm is m else a.sweep_steps,
                    "launch": "CUDA graph replay" if mm["graph"] else "plain", "clocks": mm["clocks"]}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    cpu = cpu_baseline(name, sqrt_s, seed, E, a.config) if (world == 1 and not a.no_cpu_baseline) else None

    line = {
        "metric": METRIC, "value": m["value"], "unit": "events/s", "n_gpus": world, "steps": a.steps, "warmup": a.warmup,
        "ms_per_step": m["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if a.precision == "fp64" else "f32", "data": "synthetic",
        "config": {"workload": "%s: %s, sqrt_s_hat=%g GeV, %d events/step/GPU, Philox seed %d, cuts pT>20 |eta|<2.5 dR>0.4, full %d-helicity sum"
                               % (a.config, name, sqrt_s, E, seed, info.n_hel),
                   "precision": a.precision, "l2": "flushed between steps" if m["need_flush"] else "inputs larger than L2 (%d MiB momenta)" % m["mom_mib"],
                   "parallelism": "events sharded over %d GPU(s), no collective" % world,
                   "launch": "CUDA graph replay of the 2-kernel step" if m["graph"] else "plain stream launches",
                   "why_this_config": "BASELINE.json's metric is per process and names no single config; the headline sits on the largest one "
                                      "(C5, 7 legs, 1890 diagrams, 120 colours) in FP64; every config is in per_config"},
        "roofline": {"bound": "alu", "kernel": "heget_eval_me2 (%s back end, %d-thread blocks, %d events/block, %d regs, %d B local, J in %s%s)"
                                               % (roof["kernel"], info.threads_per_block, info.events_per_block, info.regs_per_thread, info.local_bytes_per_thread,
                                                  "TMEM" if info.j_in_tmem else ("shared memory" if info.kernel == 2 else "registers/shared memory"),
                                                  ", %d warps per block of J taking turns" % info.warps_per_j if info.warps_per_j > 1 else ""),
                     "achieved": roof["achieved"], "peak": roof["peak"], "unit": "TFLOP/s", "frac": roof["frac"],
                     "executed": roof["executed"], "executed_frac": roof["executed_frac"],
                     "flop_count": "achieved = flops counted by the generator for the program it emitted (FMA = 2; scheme: %s); executed = "
                                   "ncu smsp__sass_thread_inst_executed_op_{d,f}{add,mul,fma}_pred_on per event (FMA x 2), profiles/r2_opcounts.md"
                                   % ("helicity-recycled currents, merged currents, vanishing configurations skipped" if info.kernel == 2 else "every current per configuration, vanishing configurations skipped"),
                     "traffic": TRAFFIC.get((a.config, a.precision)) if not a.events else None,
                     "traffic_note": TRAFFIC_NOTE.get((a.config, a.precision)) if not a.events else None,
                     "peak_kind": "nominal %d SMs x %d lanes x 2 x %.0f MHz (DESIGN.md)" % (SM_COUNT, FP64_LANES if a.precision == "fp64" else FP32_LANES, sm_max),
                     "fma_probe_tflops": probe, "frac_of_probe": roof["achieved"] / probe,
                     "flops_per_event": info.flops_per_event, "executed_flops_per_event": roof["executed_flops_per_event"],
                     "colour_stage": ["symmetric", "distinct", "cholesky", "tensor"][info.colour_stage] if info.kernel == 2 else "literal code",
                     "kernel_ms": m["kernel_ms"], "sampling_kernel_ms": m["sampling_ms"],
                     "kernel_share_of_step": m["kernel_ms"] / m["ms_per_step"]},
        "cpu_baseline": cpu,
        "e2e": {"value": m["e2e"], "unit": "events/s", "h2d_bytes_per_step": m["h2d"], "d2h_bytes_per_step": m["d2h"],
                "what": "heget_run_host: pinned host momenta -> device, heget_eval_me2, me2 -> pinned host, stream synchronised, per step"},
        "gpu_launches": m["launches"], "clocks": m["clocks"],
        "per_config": per_config,
        "context": {"hel_sample_events_per_s": m.get("hel_sample"),
                    "note": "one sampled helicity configuration per event, kernel only -- the mode the paper timed (BASELINE.md); not the metric"},
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C5", choices=sorted(CONFIGS))
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32", "fp32x2"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-graph", action="store_true", help="do not replay small-batch steps from a CUDA graph")
    ap.add_argument("--lanes", type=int, default=0, help="kernel variant (heget_set_lanes); 0 = automatic")
    ap.add_argument("--kernel", default=None, choices=["auto", "straight", "table"], help="kernel back end (heget_set_kernel); default automatic")
    ap.add_argument("--colour-stage", default=None, choices=["symmetric", "distinct", "cholesky", "tensor"], help="colour stage of the table back end (heget_set_colour_stage)")
    ap.add_argument("--no-sweep", action="store_true", help="skip the per_config table (every config x precision, a few steps each)")
    ap.add_argument("--sweep-steps", type=int, default=3)
    ap.add_argument("--events", type=int, default=0, help="override the events per step (ncu captures of the big configs)")
    a = ap.parse_args()
    a.warmup = max(a.warmup, 3) if a.impl == "ours" else a.warmup
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)


if __name__ == "__main__":
    main()
