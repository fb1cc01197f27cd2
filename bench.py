#!/usr/bin/env python
"""bench.py -- coupled RT + thermo-chemistry throughput on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--n 512] [--variant b]

Workload: BASELINE.json config 5 ("throughput sweep"): 512^3 coarse grid x 3 photon groups, lognormal density,
4096 sources, random x and T, seeded background radiation (variant b, so that transport does not move zeros) --
`workloads.make_config(5)`.  A "step" is one pass of the whole hot path (fused transport + chemistry pass -> chemistry
tail -> diagnostics; with --unfused: transport -> chemistry main -> tail -> diagnostics) over all cells.  `value` = cell-group updates per second, inputs resident in HBM.
`e2e` = the same metric through the C-ABI with HOST buffers: every step uploads (U, x, T) from pinned host memory
and reads (U, x, T) back.  N > 1 GPUs: independent replicas, one process per GPU.

`--impl reference` times the fp64 CPU oracle (oracle/) on the host cores on a bounded sample of the same workload.
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

METRIC = "cell_group_updates_per_s"
UNIT = "cell-group updates/s"
ORACLE_SAMPLE_N = 128             # the oracle's bounded sample of config 5: 128^3 x 3 groups (0.3 s per step on 16 cores)
ORACLE_SAMPLE_STEPS = 30          # at most this many timed steps (~10 s of host time), after the same warm-up as the GPU arm
REFERENCE_MAX_STEPS = 300         # --impl reference times exactly K steps up to this many (a few minutes of host time)
ORACLE_1T_N = 64                  # single-thread figure ("one GPU against one CPU core"): 64^3 x 3 groups
ORACLE_1T_STEPS = 8


def cpu_model():
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.lower().startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def time_oracle_single_thread(variant, warmup, config=5):
    """The same oracle with OMP_NUM_THREADS=1 (a fresh process: OpenMP reads it at start-up) on a smaller sample."""
    code = ("import sys, json; sys.path.insert(0, %r); import bench; "
            "v, secs, cores, d = bench.time_oracle(%d, %d, %d, %r, %d); print(json.dumps([v, secs, cores]))"
            % (ROOT, ORACLE_1T_N, ORACLE_1T_STEPS, warmup, variant, config))
    try:
        out = subprocess.run([sys.executable, "-c", code], env=dict(os.environ, OMP_NUM_THREADS="1"), capture_output=True,
                             text=True, timeout=600, check=True).stdout.strip().splitlines()[-1]
        v, secs, cores = json.loads(out)
        return {"value": v, "unit": UNIT, "cores": int(cores), "seconds": secs,
                "sample": "config 5%s recipe at %d^3 x 3 groups, steps %d..%d" % (variant, ORACLE_1T_N, warmup + 1, warmup + ORACLE_1T_STEPS)}
    except Exception as e:                                            # a reported baseline, never fatal
        return {"error": str(e)[:200]}


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def ncu_traffic(kernel, n):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed ncu --set full summary
    (profiles/traffic.csv; captured at 512^3) -- None for any other grid size or if no capture is recorded."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if n != (256 if kernel.startswith("amr_") else 512) or not os.path.exists(p):
        return None
    try:
        import csv
        val = None
        for row in csv.DictReader(open(p)):
            if row["kernel"] == kernel:
                val = float(row["dram_bytes_per_launch"])          # the last row of a kernel is the current capture
        return val
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except Exception:
            self.proc = None

    def _pump(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if self.proc:
            self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for ln in self.lines:
            f = [s.strip() for s in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons), "samples": len(sm)}


def time_oracle(n, steps, warmup, variant, config=5):
    """The oracle as it stands on the host cores, on config `config` at n^3 (a bounded sample of the full workload)."""
    import oracle as O
    from workloads import make_config
    w = make_config(config, n=n, variant=variant)
    orc = O.Oracle(w)
    if warmup:
        orc.step(w.dt, warmup)
    t0 = time.perf_counter()
    rc, d = orc.step(w.dt, steps)
    dt = time.perf_counter() - t0
    units = leaf_count(w) * w.G * steps
    return units / dt, dt, O.lib().orc_threads(), d


def leaf_count(w):
    """Cells that carry chemistry: every cell of every level minus the split ones (config 4; n^3 on a uniform grid)."""
    cells = [w.n ** 3] + [8 * len(p) for p in w.parent]
    split = [len(p) for p in w.parent] + [0]
    return int(sum(c - s for c, s in zip(cells, split)))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    if args.amr_standard:
        # the oracle's standard-AMR mode (serial recursion) on the same recipe at 32^3 + 2 levels
        import oracle as O
        from workloads.amr import make_amr_standard
        ws = make_amr_standard(n=32, G=3, levels=2)
        orc = O.Oracle(ws)
        assert orc.set_amr_transport(True) == O.OK
        lc = [ws.n ** 3] + [8 * len(p) for p in ws.parent]
        ll = [c - s_ for c, s_ in zip(lc, [len(p) for p in ws.parent] + [0])]
        steps, warm = max(1, min(args.steps, 6)), min(args.warmup, 1)
        if warm:
            orc.step(ws.dt, warm)
        t0 = time.perf_counter()
        orc.step(ws.dt, steps)
        secs = time.perf_counter() - t0
        val = sum(ll[l] << l for l in range(3)) * 3 * steps / secs
        sample = "standard-AMR recipe at 32^3 coarse + 2 levels x 3 groups, %d coarse steps, fp64 C oracle (serial recursion)" % steps
        line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
                "warmup": warm, "ms_per_step": 1e3 * secs / steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": "standard AMR scheme sampled at 32^3 + 2 levels (oracle on host cores)"},
                "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
                "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line), flush=True)
        return
    n = ORACLE_SAMPLE_N if args.config == 5 else 96
    # per "step" of this arm: one oracle step on the n^3 sample, timed over the SAME step range as the GPU arm (W untimed
    # warm-up steps from the seeded initial state, then EXACTLY K timed steps: ~0.3-0.8 s each on 8-16 cores, so the default
    # K = 50 takes under a minute; only a K beyond REFERENCE_MAX_STEPS is cut, and the line then says so)
    steps, warm = max(1, min(args.steps, REFERENCE_MAX_STEPS)), max(0, args.warmup)
    val, secs, cores, d = time_oracle(n, steps, warm, args.variant, args.config)
    label = ("5" + args.variant) if args.config == 5 else "4 (CRTA, 2 refined levels)"
    sample = ("config %s recipe at %d^3 x 3 groups (a bounded sample of the full grid), steps %d..%d from the seeded initial state, "
              "fp64 C oracle with OpenMP" % (label, n, warm + 1, warm + steps))
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": warm, "ms_per_step": 1e3 * secs / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": ("BASELINE config %s: %d^3 x 3 groups, coupled RT+chemistry, timed after %d warm-up steps (the GPU arm's "
                                    "workload); each step of this arm is a bounded sample of it: the same recipe at %d^3, oracle on host cores"
                                    % (label, args.n if args.config == 5 else 256, warm, n)),
                       "n_coarse": args.n if args.config == 5 else 256, "groups": 3, "sample_n_coarse": n,
                       "steps_requested": args.steps},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "cpu_model": cpu_model(), "step_range": [warm + 1, warm + steps],
                             "subcycles_mean_last_step": d["subcycles_total"] / float(n ** 3) if args.config == 5 else None},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# Issue-rate ceiling of the sub-cycling tail: SASS instructions of chem_tail_kernel<3> per accepted
# sub-step (rates at T^p 66 incl. 16 MUFU, first guess + commit + loop 64) and per attempt of Eq. 43-48 (97 incl. 4 MUFU),
# counted with cuobjdump on this build; a B200 issues 4 warp instructions per SM and clock.
TAIL_INSTR_PER_SUBSTEP = 130
TAIL_INSTR_PER_ATTEMPT = 97


def run_from_initial_state(E, torch, w, dev, K, units_per_step, sm_mhz, **kw):
    """K coupled steps from step 0 on a fresh handle, NO warm-up: the regime in which cells really sub-cycle (config 5:
    random initial T).  One step per call with its diagnostics read back, so per-step kernel times and
    sub-cycle counts are known; the host gap between steps (one 200-byte D2H + event reads) is inside the timing."""
    gpu = E.EmmaRT(w, device=dev, **kw)
    gpu.profile(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    steps = []
    torch.cuda.synchronize(dev)
    e0.record()
    for _ in range(K):
        rc, d = gpu.step(w.dt, 1, diag=True)
        assert rc == E.OK, (rc, gpu.last_error())
        steps.append((d, gpu.profile(True)))
    e1.record()
    torch.cuda.synchronize(dev)
    ms = e0.elapsed_time(e1)
    gpu.close()
    cells = units_per_step // w.G
    tail_ms = [p["chem_tail"][0] for _, p in steps]
    main_ms = [p["fused"][0] + p["chem_main"][0] + p["transport"][0] for _, p in steps]
    # evaluations of Eq. 43-48 in the tail = accepted sub-steps of the deferred cells + their rejected (halved) attempts
    sub_tail = [d["subcycles_total"] - (cells - d["n_deferred"]) for d, _ in steps]
    evals = [st + d["halvings_total"] for st, (d, _) in zip(sub_tail, steps)]
    first = [i for i in range(len(steps)) if tail_ms[i] > 0.05][:6] or [0]
    ev, tm = sum(evals[i] for i in first), sum(tail_ms[i] for i in first) * 1e-3
    instr = sum(sub_tail[i] * TAIL_INSTR_PER_SUBSTEP + evals[i] * TAIL_INSTR_PER_ATTEMPT for i in first)
    peak_lane_instr = 148 * 4 * 32 * (sm_mhz or 1965.0) * 1e6
    d1 = steps[0][0]
    return {"steps": K, "warmup": 0, "ms_per_step": ms / K, "value": units_per_step * K / (ms * 1e-3), "unit": UNIT,
            "chem_tail_ms_first_steps": [float("%.4g" % v) for v in tail_ms[:8]],
            "transport_chem_pass_ms_first_steps": [float("%.4g" % v) for v in main_ms[:8]],
            "subcycles_step1": {"mean": d1["subcycles_total"] / float(cells), "max": d1["subcycles_max"],
                                "deferred": d1["n_deferred"], "halvings": d1["halvings_total"]},
            "tail": {"steps_counted": [i + 1 for i in first], "evaluations": int(ev), "evaluations_per_s": ev / tm if tm > 0 else None,
                     "bound": "alu", "issue_ceiling_evaluations_per_s": peak_lane_instr * ev / instr if instr else None,
                     "frac_of_issue_ceiling": (instr / peak_lane_instr) / tm if tm > 0 else None,
                     "note": "ceiling = 148 SMs x 4 warp instr/clk x 32 lanes x SM clock / (130 instr per accepted sub-step + 97 "
                             "per attempt), every lane busy"}}


def run_sub_record(E, torch, w, dev, K, W, units_per_step, **kw):
    """A short device-resident run of another workload (rows a-5 / NEXT-2 of SURVEY.md section 8 at size): W warm-up steps,
    K timed ones, per-kernel CUDA-event times."""
    gpu = E.EmmaRT(w, device=dev, **kw)
    rc, _ = gpu.step(w.dt, W, diag=False)
    assert rc == E.OK, gpu.last_error()
    gpu.profile(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(dev)
    e0.record()
    rc, d = gpu.step(w.dt, K, diag=True)
    e1.record()
    torch.cuda.synchronize(dev)
    assert rc == E.OK, (rc, gpu.last_error())
    ms = e0.elapsed_time(e1)
    prof = gpu.profile(False)
    gpu.close()
    return ms, prof, d


def replica_seed(config, rank, world):
    """Seed of a rank's replica (N > 1 = independent replicas, different seeds per rank);
    None = the config's own seed (single GPU)."""
    return None if world == 1 else (150807888 + config) + 1000 * rank


def max_over_ranks(value, dist, device):
    """Device time of the job = the slowest rank's (all-reduce MAX); `dist` is torch.distributed or None."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([value], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_step, steps, world, ms):
    """Aggregate throughput of `world` replicas that each advanced `steps` steps in `ms` (max over ranks)."""
    return units_per_step * steps * world / (ms * 1e-3)


def run_ours(args):
    import torch
    import paper_1508_07888_b200 as E
    from workloads import make_config

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", local))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the library has no CPU fallback")
    torch.cuda.set_device(local)
    dev = local

    n, K, W = args.n, args.steps, args.warmup
    t0 = time.time()
    if args.config == 4 and not args.amr_standard:
        # BASELINE config 4: 256^3 coarse + 2 refined levels (CRTA); transport on the coarse level, chemistry on leaves
        w = make_config(4, n=None if n == 512 else n, seed=replica_seed(4, rank, world))
        n = w.n
        if args.boost_sources != 1.0:               # brighter sources: the refined leaves around them sub-cycle hard (row a-5)
            w.src_Q = w.src_Q * args.boost_sources
    elif args.amr_standard:
        # the standard (non-CRTA) AMR scheme on a jump-balanced config-4-like mesh
        from workloads.amr import make_amr_standard
        w = make_amr_standard(n=256 if n == 512 else n, G=3, levels=2, seed=replica_seed(4, rank, world), order=args.oct_order)
        n = w.n
    else:
        w = make_config(5, n=n, variant=args.variant, seed=replica_seed(5, rank, world))
    G = w.G
    ncell = n ** 3
    log("[bench] rank %d: generated %s in %.1f s" % (rank, w.name, time.time() - t0))

    amr = 1 if args.amr_standard else 0
    flux = E.FLUX_HLL if args.hll else None
    gpu = E.EmmaRT(w, device=dev, fused=0 if args.unfused else 1, amr_transport=amr, flux=flux)
    dt = w.dt
    units_per_step = leaf_count(w) * G            # config 5: n^3 G; config 4: leaf cells x G
    lv_cells = [n ** 3] + [8 * len(p) for p in w.parent]
    lv_leaves = [c - s for c, s in zip(lv_cells, [len(p) for p in w.parent] + [0])]
    if amr:                                       # a level-l leaf is advanced 2^l times per coarse step (dt_l = dt/2^l)
        units_per_step = sum(lv_leaves[l] << l for l in range(len(lv_leaves))) * G

    def barrier():
        torch.cuda.synchronize(dev)
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize(dev)

    # ---------------- device-resident: W warm-up steps, then exactly K timed steps
    rc, _ = gpu.step(dt, W, diag=False)
    assert rc == E.OK, gpu.last_error()
    gpu.profile(True)
    launches0 = gpu.kernel_launches()
    clocks = ClockSampler(dev)
    clocks.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    rc, diag = gpu.step(dt, K, diag=True)
    e1.record()
    barrier()
    clk = clocks.stop()
    assert rc == E.OK, (rc, gpu.last_error())
    ms = e0.elapsed_time(e1)
    launches = gpu.kernel_launches() - launches0
    prof = gpu.profile(False)
    ms = max_over_ranks(ms, dist, "cuda")
    value = whole_job_value(units_per_step, K, world, ms)

    # per-kernel roofline (algorithmic bytes of DESIGN.md section 7 / live CUDA-event durations)
    peak, peak_src = measured_peaks()
    alg = {"transport": 32.0 * ncell * G,                    # 16 B read + 16 B write per cell-group
           "chem_main": (32.0 * G + 20.0) * ncell,           # U in/out + n0, x, e in + x, e out per cell
           "fused": (32.0 * G + 20.0) * ncell}               # single pass: U in, U out, n0, x, e in, x, e out
    # refined-level sweeps of the standard AMR scheme: bytes of all the sweeps of one coarse step (levels >= 1)
    alg_step = {"amr_transport": 32.0 * G * sum(lv_leaves[l] << l for l in range(1, len(lv_leaves))),
                "amr_chem": (32.0 * G + 20.0) * sum(lv_leaves[l] << l for l in range(1, len(lv_leaves)))}
    kern = {}
    for k, (kms, cnt) in prof.items():
        if cnt:
            kern[k] = {"ms_per_launch": kms / cnt, "launches": int(cnt), "share": kms / ms}
            if k in alg_step and amr:
                kern[k]["GBps"] = alg_step[k] * K / (kms * 1e-3) / 1e9
                kern[k]["frac"] = kern[k]["GBps"] / peak
                alg[k] = alg_step[k] * K / cnt
            elif k in alg:
                kern[k]["GBps"] = alg[k] / (kms / cnt * 1e-3) / 1e9
                kern[k]["frac"] = kern[k]["GBps"] / peak
    dominant = max((k for k in kern if k in alg), key=lambda k: kern[k]["share"])
    roofline = {"kernel": dominant, "bound": "hbm", "achieved": kern[dominant]["GBps"], "peak": peak, "unit": "GB/s",
                "frac": kern[dominant]["frac"], "traffic": None, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg[dominant]}
    roofline["traffic"] = ncu_traffic(dominant, n)

    # ---------------- transport-only throughput (chemistry = 0), same grid, K steps
    tr = hll = None
    if not args.skip_transport_only and not amr:
        gpu.close()
        gpu = None
        torch.cuda.empty_cache()
        g2 = E.EmmaRT(w, device=dev, chemistry=0)
        g2.step(dt, W, diag=False)
        barrier()
        e0.record()
        g2.step(dt, K, diag=False)
        e1.record()
        barrier()
        ms_t = e0.elapsed_time(e1)
        tr = {"value": ncell * G * K / (ms_t * 1e-3), "unit": UNIT, "ms_per_step": ms_t / K,       # coarse cells x G
              "GBps": 32.0 * ncell * G * K / (ms_t * 1e-3) / 1e9}
        tr["frac"] = tr["GBps"] / peak
        g2.close()
        torch.cuda.empty_cache()
        # the same with the HLL interface flux (emma_rt_set_flux)
        g3 = E.EmmaRT(w, device=dev, chemistry=0, flux=E.FLUX_HLL)
        g3.step(dt, W, diag=False)
        barrier()
        e0.record()
        g3.step(dt, K, diag=False)
        e1.record()
        barrier()
        ms_h = e0.elapsed_time(e1)
        hll = {"value": ncell * G * K / (ms_h * 1e-3), "unit": UNIT, "ms_per_step": ms_h / K,
               "GBps": 32.0 * ncell * G * K / (ms_h * 1e-3) / 1e9}
        hll["frac"] = hll["GBps"] / peak
        g3.close()
        torch.cuda.empty_cache()
        gpu = E.EmmaRT(w, device=dev, fused=0 if args.unfused else 1, amr_transport=amr, flux=flux)

    # ---------------- the hard regime: the same workload from the seeded initial state, no warm-up (sub-cycling transient)
    init_leg = None
    if args.config == 5 and not amr and not args.skip_initial_state:
        if gpu is not None:
            gpu.close()
            gpu = None
            torch.cuda.empty_cache()
        init_leg = run_from_initial_state(E, torch, w, dev, K, units_per_step, clk.get("sm_mhz"),
                                          fused=0 if args.unfused else 1, flux=flux)
        gpu = E.EmmaRT(w, device=dev, fused=0 if args.unfused else 1, amr_transport=amr, flux=flux)

    # ---------------- rows a-5 (CRTA, BASELINE config 4) and NEXT-2 (standard AMR) at size, as short sub-records
    extra = {}
    if args.config == 5 and not amr and not args.skip_extra and world == 1:
        gpu.close()
        gpu = None
        torch.cuda.empty_cache()
        try:
            w4 = make_config(4)
            u4 = leaf_count(w4) * w4.G
            ms4, p4, d4 = run_sub_record(E, torch, w4, dev, min(K, 20), W, u4)
            extra["config4_crta"] = {
                "workload": "BASELINE config 4: 256^3 coarse + 2 refined levels (CRTA), 3 groups, %d leaves, %d sources" % (leaf_count(w4), len(w4.src_pos)),
                "steps": min(K, 20), "warmup": W, "ms_per_step": ms4 / min(K, 20), "value": u4 * min(K, 20) / (ms4 * 1e-3),
                "unit": "leaf-" + UNIT, "kernels_ms_per_step": {k: v[0] / min(K, 20) for k, v in p4.items() if v[1]},
                "subcycles_max_last_step": d4["subcycles_max"], "deferred_last_step": d4["n_deferred"]}
            del w4
        except Exception as e:                                        # a sub-record never costs the headline line
            extra["config4_crta"] = {"error": str(e)[:300]}
        try:
            from workloads.amr import make_amr_standard
            wa = make_amr_standard(n=256, G=3, levels=2)
            ca = [wa.n ** 3] + [8 * len(p) for p in wa.parent]
            la = [c - s_ for c, s_ in zip(ca, [len(p) for p in wa.parent] + [0])]
            ua = sum(la[l] << l for l in range(3)) * wa.G
            Ka = min(K, 10)
            msa, pa, da = run_sub_record(E, torch, wa, dev, Ka, W, ua, amr_transport=1)
            ref_sweeps = sum(la[l] << l for l in range(1, 3))
            extra["amr_standard"] = {
                "workload": "standard AMR scheme (SURVEY 8f NEXT-2, reading A21): 256^3 + 2 refined levels, 3 groups, cells per level %s, "
                            "leaves per level %s; a level-l leaf counts 2^l times per coarse step" % (ca, la),
                "steps": Ka, "warmup": W, "ms_per_step": msa / Ka, "value": ua * Ka / (msa * 1e-3), "unit": "leaf-" + UNIT,
                "kernels_ms_per_step": {k: v[0] / Ka for k, v in pa.items() if v[1]},
                "amr_transport": {"algorithmic_bytes_per_step": 32.0 * wa.G * ref_sweeps,
                                  "GBps": 32.0 * wa.G * ref_sweeps * Ka / (pa["amr_transport"][0] * 1e-3) / 1e9,
                                  "frac": 32.0 * wa.G * ref_sweeps * Ka / (pa["amr_transport"][0] * 1e-3) / 1e9 / peak}}
            del wa
        except Exception as e:
            extra["amr_standard"] = {"error": str(e)[:300]}
        torch.cuda.empty_cache()
        gpu = E.EmmaRT(w, device=dev, fused=0 if args.unfused else 1, amr_transport=amr, flux=flux)

    # ---------------- end to end through the C-ABI with host buffers (pinned), copies inside the timed region
    Ke = max(1, min(K, args.e2e_steps))
    hU = [torch.from_numpy(np.ascontiguousarray(w.U0[g])).pin_memory() if w.U0 is not None
          else torch.zeros((ncell, 4), dtype=torch.float32).pin_memory() for g in range(G)]
    hx = torch.from_numpy(w.x[0].copy()).pin_memory()
    hT = torch.from_numpy(w.T[0].copy()).pin_memory()
    h2d = sum(t.numel() * 4 for t in hU) + hx.numel() * 4 + hT.numel() * 4
    d2h = h2d

    use_host = args.config == 5 and not amr and not args.unfused and not args.hll

    def e2e_serial():
        for g in range(G):
            assert gpu.write(E.FIELD_U, 0, g, hU[g]) == E.OK
        assert gpu.write(E.FIELD_X, 0, 0, hx) == E.OK
        assert gpu.write(E.FIELD_T, 0, 0, hT) == E.OK
        rc, _ = gpu.step(dt, 1, diag=False)
        assert rc == E.OK
        for g in range(G):
            assert gpu.read_into(E.FIELD_U, 0, g, hU[g]) == E.OK
        assert gpu.read_into(E.FIELD_X, 0, 0, hx) == E.OK
        assert gpu.read_into(E.FIELD_T, 0, 0, hT) == E.OK

    def e2e_step():
        if use_host:                                              # host state in, host state out, slab-pipelined (one C-ABI call)
            rc, _ = gpu.step_host(dt, hU, hx, hT, diag=False)
            assert rc == E.OK, gpu.last_error()
        else:
            e2e_serial()

    e2e_step()                                                # warm-up (page-locks, first-touch)
    barrier()
    t0 = time.perf_counter()
    for _ in range(Ke):
        e2e_step()
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, dist, "cuda")
    e2e = {"value": units_per_step * Ke * world / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h, "steps": Ke, "ms_per_step": 1e3 * e2e_s / Ke,
           "api": "emma_rt_step_host (z-slab pipeline: H2D, fused pass, D2H on three streams)" if use_host
                  else "emma_rt_write x5 -> emma_rt_step -> emma_rt_read x5",
           "link_GBps_each_way": h2d / (e2e_s / Ke) / 1e9}
    if use_host:                                                  # the same bytes through the serial calls, for comparison
        barrier()
        t0 = time.perf_counter()
        for _ in range(2):
            e2e_serial()
        barrier()
        e2e["serial_write_step_read_ms_per_step"] = 1e3 * (time.perf_counter() - t0) / 2
    gpu.close()

    # ---------------- oracle on the host cores, bounded sample (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.skip_cpu_baseline and amr:
        import oracle as O
        from workloads.amr import make_amr_standard
        ws = make_amr_standard(n=32, G=3, levels=2)
        orc = O.Oracle(ws)
        assert orc.set_amr_transport(True) == O.OK
        lc = [ws.n ** 3] + [8 * len(p) for p in ws.parent]
        ll = [c - s_ for c, s_ in zip(lc, [len(p) for p in ws.parent] + [0])]
        t0 = time.perf_counter()
        orc.step(ws.dt, 6)
        secs = time.perf_counter() - t0
        cpu = {"value": sum(ll[l] << l for l in range(3)) * 3 * 6 / secs, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": secs,
               "sample": "standard-AMR recipe at 32^3 coarse + 2 levels x 3 groups, 6 coarse steps, fp64 C oracle (the AMR "
                         "recursion of the oracle is serial)"}
    elif rank == 0 and world == 1 and not args.skip_cpu_baseline:
        osteps = max(1, min(K, ORACLE_SAMPLE_STEPS))
        on = ORACLE_SAMPLE_N if args.config == 5 else 96
        val, secs, cores, od = time_oracle(on, osteps, W, args.variant, args.config)
        cpu = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": secs, "cpu_model": cpu_model(),
               "step_range": [W + 1, W + osteps],
               "sample": "config %s recipe at %d^3 x 3 groups, steps %d..%d from the seeded initial state (the GPU arm's timed "
                         "range: %d warm-up steps first), fp64 C oracle as it stands, OpenMP on all host cores"
                         % ("5" + args.variant if args.config == 5 else "4 (CRTA, 2 levels)", on, W + 1, W + osteps, W),
               # the paper's own convention is one graphics device against ONE CPU core
               "single_thread": time_oracle_single_thread(args.variant, W) if args.config == 5 else None}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
                "data": "synthetic",
                "config": {"workload": ("BASELINE config 5%s: %d^3 x %d groups, lognormal sigma_ln=1.0, %d sources, "
                                        "random x,T, coupled RT+chemistry; STEADY STATE: timed after %d warm-up steps, ~%.3f accepted "
                                        "sub-steps per cell (the sub-cycling transient of the random initial T falls in the warm-up: "
                                        "see coupled_from_initial_state for the same workload from step 0)"
                                        % (args.variant, n, G, len(w.src_pos), W, diag["subcycles_total"] / float(leaf_count(w))))
                           if args.config == 5 and not amr else
                           ("standard AMR scheme (SURVEY 8f NEXT-2, reading A21): %d^3 coarse + 2 refined levels on a jump-balanced "
                            "config-4-like mesh, %d groups, cells per level %s, leaves per level %s, %d sources; value counts "
                            "leaf-cell-group updates, a level-l leaf 2^l times per coarse step" % (n, G, lv_cells, lv_leaves, len(w.src_pos)))
                           if amr else
                           ("BASELINE config 4: %d^3 coarse + 2 refined levels (CRTA), %d groups, lognormal sigma_ln=1.5, "
                            "%d leaves, %d sources; value counts leaf-cell-group updates" % (n, G, leaf_count(w), len(w.src_pos))),
                           "n_coarse": n, "groups": G, "cells": ncell, "dt_s": dt, "l2": "inputs_exceed_l2",
                           "schedule": "unfused" if (args.unfused or args.hll or amr) else "fused",
                           "flux": "hll" if args.hll else "glf",
                           "parallelism": "replicas" if world > 1 else "single"},
                "roofline": roofline, "kernels": kern, "transport_only": tr, "transport_only_hll": hll, "e2e": e2e, "cpu_baseline": cpu,
                "coupled_from_initial_state": init_leg, "sub_records": extra or None,
                "gpu_launches": int(launches), "clocks": clk,
                "subcycles": {"mean_last_step": diag["subcycles_total"] / float(leaf_count(w)), "max_last_step": diag["subcycles_max"],
                              "deferred_last_step": diag["n_deferred"]}}
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=512)
    ap.add_argument("--variant", default="b", choices=["a", "b"])
    ap.add_argument("--config", type=int, default=5, choices=[4, 5], help="BASELINE config: 5 (default, the metric's) or 4 (CRTA)")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--unfused", action="store_true", help="separate transport and chemistry passes")
    ap.add_argument("--oct-order", default="id", choices=["id", "morton"],
                    help="memory order of the octs of --amr-standard: parent-cell id, or Z-order of the parent's coordinates")
    ap.add_argument("--hll", action="store_true", help="coupled step with the HLL interface flux (two-pass schedule)")
    ap.add_argument("--amr-standard", action="store_true",
                    help="the standard (non-CRTA) AMR scheme on a jump-balanced 256^3 + 2 levels mesh (SURVEY 8f NEXT-2)")
    ap.add_argument("--skip-transport-only", action="store_true")
    ap.add_argument("--skip-cpu-baseline", action="store_true")
    ap.add_argument("--skip-initial-state", action="store_true", help="skip the no-warm-up leg (coupled_from_initial_state)")
    ap.add_argument("--boost-sources", type=float, default=1.0, help="--config 4 only: multiply every source's Q (divergent sub-cycling on the refined levels)")
    ap.add_argument("--skip-extra", action="store_true", help="skip the config-4 (CRTA) and standard-AMR sub-records")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
