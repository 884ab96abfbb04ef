"""bench.py -- throughput of the EPRL vertex-tensor hot path (all rows of SURVEY.md 8(a)) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference] [--path 0..4]

A "step" is one pass of the whole hot path over one workload: one sf_vertex_amplitude call (k-range tables, the five S
arrays of {6j}, {15j} assembly + four mode products over every shell, fixed-order accumulation, normalisation).  The
default workload is config 3 of BASELINE.json (all spins j = 5, Delta_l = 10: 1 771 561 shells, A[11^5]), the
configuration the headline metric is quoted on.  The {6j} table (sf_sixj_table, a one-off like the paper's precomputed
tables) is built before the timed region and reported separately.

N > 1: the path does not shard (north_star: one GPU, no collectives) => N independent replicas, one per rank,
"scaling": "weak"; value = shells of all replicas / max-over-ranks time.

The library takes the fastest path that holds the problem (`--path 0`): the factorised path (the sum of eq. (3) taken one
virtual spin at a time, DESIGN.md 5 K-f); `--path 3` times the per-shell line kernel instead.  Timed region: K asynchronous
calls between two CUDA events on the call's stream.  `roofline` then comes from a second, instrumented pass of K steps
(per-kernel CUDA events inside the library): achieved = USEFUL FP64 flop of the kernel that takes the most time (multiply-
adds on the index combinations the triangle inequalities allow, counted on the host by sf_factor_work: no tile padding, no
window rounding) / its event time, against the DMMA peak measured in this process.  The executed DMMA count (padding
included, from the kernels' own counters) is reported beside it as `executed_over_useful`, never as the fraction.  Because
the factorised sum is not the per-shell method of the paper, `value` on that path is a shells-EQUIVALENT rate (nominal
shells of the tensor / time); the per-shell method itself (`--path 3`, SURVEY.md 8(d)'s F_asm + F_con) is timed in the same
run and reported as `per_shell_path`.

Prints ONE JSON line (rank 0).  `--impl reference` times the oracle (oracle/, plain CPU loops) on the host cores on a
bounded sample of the same workload.
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

import workloads as wl  # noqa: E402

METRIC = "eprl_shells_contracted_per_s"
PATH_NAMES = {1: "staged", 3: "line", 4: "factorised"}
# DRAM traffic per launch comes from the committed ncu launch list of one config-3 step (every kernel of one
# sf_vertex_amplitude call with dram__bytes_read.sum, dram__bytes_write.sum, gpu__time_duration.sum); null for other workloads
NCU_LAUNCHES_CONFIG3 = os.path.join("profiles", "r3_config3_step_launches.csv")
FZ_KERNELS = {"qp": ("k_fz_qp",), "R": ("k_fz_r3", "k_fz_r2", "k_fz_gemm<FzMapR"), "A": ("k_fz_gemm<FzMapA",)}
UNIT = "shells/s"


def workload(config, sub):
    if config == 0:
        return wl.CONFIGS[0]
    if config == 2:
        return wl.config2(sub if sub is not None else 8)
    if config == 3:
        return wl.CONFIGS[3]
    raise SystemExit("bench workloads: --config 0, 2 (with --sub DELTA_L) or 3")


# ---------------------------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md recipe)
# ---------------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
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
            self.rows.append((time.perf_counter(), [c.strip() for c in line.split(",")]))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for t, r in self.rows if t0 <= t <= t1] or [r for _, r in self.rows[-3:]]
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); smax.append(float(r[1])); power.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------------------------
# CPU baseline = the oracle as it stands, on a bounded sample of the workload
# ---------------------------------------------------------------------------------------------------------------
def oracle_sample(cfg, B, n_sample, seed=12345):
    """(lo, hi, S arrays): a seeded contiguous range of `n_sample` shells and the exact-{6j} S arrays it needs (the
    paper also precomputes its {6j} tables; not timed)."""
    from oracle import vertex as ov
    L = ov.Layout(cfg["two_j"], cfg["two_dl"])
    n_sample = min(n_sample, L.n_shells)
    rng = np.random.Generator(np.random.PCG64(seed))
    lo = int(rng.integers(0, L.n_shells - n_sample + 1))
    S = ov.build_s_arrays(L, lo, lo + n_sample, processes=os.cpu_count() or 1)
    return lo, lo + n_sample, S


def oracle_time(cfg, B, lo, hi, S, threads):
    from oracle import vertex as ov
    t0 = time.perf_counter()
    r = ov.vertex_l1(cfg["two_j"], cfg["two_dl"], B, shell_lo=lo, shell_hi=hi, long_double=False, want_abs=False,
                     threads=threads, s_arrays=S)
    return time.perf_counter() - t0, r


def dims_from_oracle(cfg):
    from oracle import ranges
    edge_dims, k_ranges = {}, {}
    for edge in (2, 3, 4, 5):
        _, n_i, _, base, pad = ranges.booster_dims(cfg["two_j"], cfg["two_dl"], edge)
        edge_dims[edge] = (n_i, base, pad)
        k_ranges[edge] = ranges.booster_k_ranges(cfg["two_j"], cfg["two_dl"], edge)
    return edge_dims, k_ranges


def run_reference(args, cfg, rank):
    """The oracle as it stands on the host cores: each step = one bounded sample of the workload's shells."""
    if rank != 0:
        return
    edge_dims, k_ranges = dims_from_oracle(cfg)
    nl = cfg["two_dl"] // 2 + 1
    B = wl.random_boosters(cfg["seed"], nl, edge_dims, k_ranges)
    cores = os.cpu_count() or 1
    n_sample = min(args.ref_shells, nl ** 6)
    lo, hi, S = oracle_sample(cfg, B, n_sample)
    for _ in range(args.warmup):
        oracle_time(cfg, B, lo, min(hi, lo + max(1, n_sample // 8)), S, cores)
    total = 0.0
    for _ in range(args.steps):
        dt, _ = oracle_time(cfg, B, lo, hi, S, cores)
        total += dt
    value = (hi - lo) * args.steps / total
    sample = f"shells [{lo},{hi}) of {nl ** 6} per step (seeded contiguous range), exact-6j S arrays precomputed untimed"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "two_j": cfg["two_j"], "two_dl": cfg["two_dl"], "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def max_over_ranks(values, world, device):
    """Element-wise maximum of per-rank timings over all ranks (replicas: the job takes as long as its slowest rank)."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def whole_job_value(units_per_rank, steps, world, seconds):
    """Whole-job throughput of `world` replicas that each processed `units_per_rank` units per step."""
    return world * units_per_rank * steps / seconds


def bench_contractions(torch, sf, stream):
    """Secondary row (SURVEY.md K-e; Fig. 3): vertex x vertex and vertex x five complex vectors on
    synthetic tensors of (2J+1)^5 entries, J = 10 and J = 20.  HBM-bound streaming reductions: algorithmic bytes = 8 B per
    entry read once (16 B for two tensors) / CUDA-event time, against the measured copy bandwidth."""
    peak = None
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            peak = float(json.load(fh)["hbm_gbs"])
    except (OSError, KeyError, ValueError):
        pass
    peak_src = "MEASURED_PEAKS.json hbm_gbs" if peak else "fallback of B200_PROFILING.md (6550 GB/s copy bandwidth)"
    peak = peak or 6550.0
    out = {"unit": "GB/s", "peak": peak, "peak_source": peak_src, "bound": "hbm", "cases": []}
    for n in (21, 41):
        A = torch.randn((n,) * 5, dtype=torch.float64, device="cuda")
        B = torch.randn((n,) * 5, dtype=torch.float64, device="cuda")
        psi = [torch.randn(n, dtype=torch.complex128, device="cuda") for _ in range(5)]
        res = torch.zeros(2, dtype=torch.float64, device="cuda")
        for name, call, nbytes in (("vertex_x_vertex", lambda: sf.sf_contract_vertices(A, B, res, stream), 16 * A.numel()),
                                   ("vertex_x_5_vectors", lambda: sf.sf_contract_vectors(A, psi, res, stream), 8 * A.numel())):
            for _ in range(3):
                call()
            reps = 20
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(reps):
                call()
            e1.record(stream)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / reps
            gbs = nbytes / (ms * 1e-3) / 1e9
            out["cases"].append({"contraction": name, "entries": A.numel(), "ms": ms, "achieved": gbs, "frac": gbs / peak,
                                 "note": "back-to-back repeats: the %d MB working set %s the 126 MB L2"
                                         % (nbytes >> 20, "fits" if nbytes < 126 << 20 else "exceeds")})
        del A, B
    return out


def bench_other_workloads(torch, sf, stream, peak):
    """The other four workloads of BASELINE.json in full (north_star: throughput on all five), each a few asynchronous calls
    between two CUDA events: config 0, config 1 at j = 10 (identity boosters, A = N(i) {15j}), config 2 at Delta_l = 8,
    config 4 at lambda = 1..6.  Secondary rows: the headline stays config 3."""
    def valid(two_j):
        try:
            sf.sf_vertex_dims(two_j)
            return True
        except sf.SfError:
            return False

    base, _ = wl.config4_base_spins(valid)
    cases = [wl.CONFIGS[0], wl.config1(20), wl.config2(8)] + [wl.config4(base, lam) for lam in range(1, 7)]
    rows = []
    for c in cases:
        two_j, two_dl = c["two_j"], c["two_dl"]
        nl = two_dl // 2 + 1
        edge_dims, k_ranges = {}, {}
        for edge in (2, 3, 4, 5):
            _, n_i_e, kbase, pad = sf.sf_booster_dims(two_j, two_dl, edge)
            edge_dims[edge] = (n_i_e, kbase, pad)
            k_ranges[edge] = sf.sf_booster_kranges(two_j, two_dl, edge)
        lo, n_i = sf.sf_vertex_dims(two_j)
        if c["boosters"] == "identity":
            B = wl.identity_boosters(edge_dims, lo)
        else:
            B = wl.random_boosters(c["seed"], nl, edge_dims, k_ranges)
        Bdev = [torch.from_numpy(np.ascontiguousarray(B[e])).cuda() for e in (2, 3, 4, 5)]
        out = torch.zeros(tuple(n_i), dtype=torch.float64, device="cuda")
        for _ in range(4):              # warm-up: sizes the scratch buffers; the third identical call records the launch sequence
            sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, stream)      # (sf_set_graphs, include/sfoam.h), later ones replay it
        torch.cuda.synchronize()
        reps = 10 if nl ** 6 * int(np.prod(n_i)) < 10 ** 10 else 2
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, stream)
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / reps
        row = {"workload": c["name"], "shells": nl ** 6, "out_shape": list(n_i), "ms_per_tensor": ms,
               "shells_equivalent_per_s": nl ** 6 / (ms * 1e-3), "tensors_per_s": 1e3 / ms,
               "path": PATH_NAMES.get(sf.sf_last_path(), "?"), "finite": bool(torch.isfinite(out).all())}
        if sf.sf_last_path() == 4:      # roofline fraction of the whole call on the useful flop of the factorised chain
            flop, _, _ = factor_work(sf, two_j, two_dl)
            useful = sum(flop.values())
            row["useful_flop"] = useful
            row["useful_tflops"] = useful / (ms * 1e-3) / 1e12
            row["frac"] = row["useful_tflops"] / peak
            row["limiter"] = ("launch latency (about 20 dependent graph nodes per call)" if ms < 0.3 else
                              "FP64 tensor pipe (alu) with operand latency, see roofline.kernels")
        rows.append(row)
        del Bdev, out
    return rows



def hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except (OSError, KeyError, ValueError):
        return 6550.0, "fallback of B200_PROFILING.md (6550 GB/s copy bandwidth)"


def ncu_dram_per_step():
    """{kernel class: (launches, bytes)} and the total, summed over all launches of one config-3 step, from the committed ncu
    launch list (profiles/r3_config3_step_launches.csv: one row per launch and metric).  None if the file is absent."""
    import csv
    path = os.path.join(ROOT, NCU_LAUNCHES_CONFIG3)
    if not os.path.exists(path):
        return None
    per, total = {}, 0.0
    with open(path) as fh:
        rows = [r for r in csv.reader(fh) if len(r) > 5]
    head = next((r for r in rows if "Kernel Name" in r), None)
    if head is None:
        return None
    k_name, k_metric, k_unit, k_val, k_id = (head.index(c) for c in ("Kernel Name", "Metric Name", "Metric Unit", "Metric Value", "ID"))
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    seen = {}
    for r in rows:
        if r is head or not r[k_metric].startswith("dram__bytes_"):
            continue
        b = float(r[k_val].replace(",", "")) * scale.get(r[k_unit], 1.0)
        name = r[k_name].split("(")[0].replace("void ", "")
        if not name.startswith(("k_fz_", "k_slices", "k_kranges")):
            continue                                  # the one-off {6j} table build is not part of a step
        cls = next((c for c, pats in FZ_KERNELS.items() if name.startswith(pats)), "other")
        n, tot = per.get(cls, (0, 0.0))
        seen.setdefault(cls, set()).add(r[k_id])
        per[cls] = (len(seen[cls]), tot + b)
        total += b
    return {"per_kernel": {c: {"launches": n, "bytes": b} for c, (n, b) in per.items()}, "total": total,
            "source": NCU_LAUNCHES_CONFIG3}


def factor_work(sf, two_j, two_dl):
    """Useful flop of the factorised chain per kernel (host integer count, include/sfoam_debug.h) and the algorithmic bytes
    of its intermediates (every structurally non-zero entry of P and R written once and read once, 8 B each)."""
    mac, elems = sf.sf_factor_work(two_j, two_dl)
    flop = {"qp": 2.0 * (mac["Q"] + mac["P"]), "R": 2.0 * mac["R"], "A": 2.0 * mac["A"], "pre": 2.0 * (mac["Z"] + mac["G"])}
    return flop, mac, elems


def bench_many_vertices(torch, sf, stream, n=1024):
    """SURVEY.md 8(f) item 1 ("many vertex tensors with few shells"): n config-0 vertex tensors (all spins 1,
    Delta_l = 2, 729 shells each) through sf_vertex_amplitude_batch -- one kernel launch, one CTA per tensor -- against n
    single calls; CUDA events on the stream, the {6j} table of the bench resident."""
    cfg = wl.CONFIGS[0]
    two_j, two_dl = cfg["two_j"], cfg["two_dl"]
    nl = two_dl // 2 + 1
    edge_dims, k_ranges = {}, {}
    for edge in (2, 3, 4, 5):
        _, n_i_e, kbase, pad = sf.sf_booster_dims(two_j, two_dl, edge)
        edge_dims[edge] = (n_i_e, kbase, pad)
        k_ranges[edge] = sf.sf_booster_kranges(two_j, two_dl, edge)
    _, n_i = sf.sf_vertex_dims(two_j)
    Bs, outs = [], []
    for q in range(n):                                # every tensor has its own boosters (seeded) and its own output
        B = wl.random_boosters(cfg["seed"] + q, nl, edge_dims, k_ranges)
        Bs.append([torch.from_numpy(np.ascontiguousarray(B[e])).cuda() for e in (2, 3, 4, 5)])
        outs.append(torch.zeros(tuple(n_i), dtype=torch.float64, device="cuda"))
    spins = [two_j] * n
    for _ in range(3):
        sf.sf_vertex_amplitude_batch(spins, two_dl, Bs, outs, stream)
    torch.cuda.synchronize()
    sf.sf_launch_count(reset=True)
    reps = 5
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(reps):
        sf.sf_vertex_amplitude_batch(spins, two_dl, Bs, outs, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    launches = sf.sf_launch_count() // reps
    ref = torch.zeros(tuple(n_i), dtype=torch.float64, device="cuda")
    sf.sf_vertex_amplitude(two_j, two_dl, Bs[7], ref, stream)
    torch.cuda.synchronize()
    m = 64
    e0.record(stream)
    for q in range(m):
        sf.sf_vertex_amplitude(two_j, two_dl, Bs[q], outs[q], stream)
    e1.record(stream)
    torch.cuda.synchronize()
    single_ms = e0.elapsed_time(e1) / m
    sf.sf_vertex_amplitude_batch(spins, two_dl, Bs, outs, stream)
    torch.cuda.synchronize()
    return {"workload": f"{n} x {cfg['name']}", "tensors": n, "ms_per_batch": ms, "tensors_per_s": n / (ms * 1e-3),
            "launches_per_batch": launches, "single_call_ms_per_tensor": single_ms,
            "single_call_tensors_per_s": 1e3 / single_ms, "speedup_over_single_calls": single_ms * n / ms,
            "max_abs_diff_vs_single_over_max": float((outs[7] - ref).abs().max() / ref.abs().max()),
            "kernel": "k_vertex_batch (one CTA per tensor; FP64 FMA, S arrays and all intermediates in shared memory)",
            "limiter": "instruction issue / shared-memory latency: index arithmetic of the irregular ranges dominates the "
                       "3.4e6 flop per tensor"}


def run_ours(args, cfg, rank, world, local_rank):
    import torch
    import torch.distributed as dist

    import paper_2107_13952_b200 as sf

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    two_j, two_dl = cfg["two_j"], cfg["two_dl"]
    nl = two_dl // 2 + 1
    n_shells = nl ** 6

    sf.sf_init(wl.GAMMA)
    sf.sf_set_path(args.path)
    if args.variant:
        sf.sf_set_factor_variant(args.variant)       # A/B timing of the factorised kernels (include/sfoam_debug.h)
    # one-off {6j} table (kernel (a)), outside the timed region, timed on its own
    t0 = time.perf_counter()
    sf.sf_sixj_table(args.table)
    torch.cuda.synchronize()
    table_ms = 1e3 * (time.perf_counter() - t0)

    edge_dims, k_ranges = {}, {}
    for edge in (2, 3, 4, 5):
        _, n_i_e, base, pad = sf.sf_booster_dims(two_j, two_dl, edge)
        edge_dims[edge] = (n_i_e, base, pad)
        k_ranges[edge] = sf.sf_booster_kranges(two_j, two_dl, edge)
    B = wl.random_boosters(cfg["seed"], nl, edge_dims, k_ranges)
    Bhost = [torch.from_numpy(B[e]).pin_memory() for e in (2, 3, 4, 5)]
    Bdev = [b.cuda() for b in Bhost]
    _, n_i = sf.sf_vertex_dims(two_j)
    out = torch.zeros(tuple(n_i), dtype=torch.float64, device="cuda")
    out_host = torch.zeros(tuple(n_i), dtype=torch.float64).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    stream = torch.cuda.current_stream()

    # algorithmic work (valid ranges only): host integer count of the contraction, device integer count of eq. (5) terms
    work = sf.sf_vertex_work(two_j, two_dl)
    n_terms = sf.sf_vertex_terms(two_j, two_dl)
    f_con, f_asm = work["f_con"], 6.0 * n_terms

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.one_step_only:      # profiling aid: the {6j} table build and exactly one vertex call, nothing else (ncu launch lists)
        sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, stream)
        torch.cuda.synchronize()
        if rank == 0:
            print(json.dumps({"one_step_only": True, "workload": cfg["name"], "path": PATH_NAMES.get(sf.sf_last_path(), "?"),
                              "gpu_launches": sf.sf_launch_count(), "max_abs": float(out.abs().max())}))
        return
    for _ in range(args.warmup):
        flush.zero_()
        sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, stream)
    torch.cuda.synchronize()

    # ---- timed region: K steps, inputs resident in HBM; the calls are asynchronous, nothing but CUDA events in it ----
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.3)
    sf.sf_launch_count(reset=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    w0 = time.perf_counter()
    e0.record(stream)
    for _ in range(args.steps):
        flush.zero_()
        sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, stream)
    e1.record(stream)
    barrier()
    w1 = time.perf_counter()
    launches = sf.sf_launch_count()
    clocks = sampler.stop(w0, w1)
    ms = e0.elapsed_time(e1)
    # ---- the same K steps again with the library's own CUDA events on (per stage, per kernel): each call then ends with a
    #      stream synchronise, so these steps are not the ones `value` is computed from ----
    sf.sf_set_timing(True)
    stage = np.zeros(3)
    kms = np.zeros(4)                 # factorised path: event times of its kernels (k_fz_qp, R, A', precomputations)
    for _ in range(args.steps):
        flush.zero_()
        sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, stream)
        stage += np.array(sf.sf_last_stage_ms())
        kms += np.array(sf.sf_last_kernel_ms())
    sf.sf_set_timing(False)
    last_path = sf.sf_last_path()
    A_dev = out.cpu().numpy().copy()
    dmma = [0.0, 0.0, 0.0]
    if last_path == 4:                # one untimed call with the kernels' DMMA counters on (the executed work)
        sf.sf_set_counting(True)
        sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, stream)
        dmma = sf.sf_last_dmma()
        sf.sf_set_counting(False)
        assert np.array_equal(out.cpu().numpy(), A_dev), "counting changed the result"

    # ---- end to end: host buffers in, host tensor out, through sf_vertex_amplitude_host ----
    for _ in range(min(args.warmup, 2)):
        sf.sf_vertex_amplitude_host(two_j, two_dl, Bhost, out_host, stream)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        flush.zero_()
        sf.sf_vertex_amplitude_host(two_j, two_dl, Bhost, out_host, stream)      # synchronises `stream` itself
    barrier()
    e2e_s = time.perf_counter() - t0
    h2d = int(sum(b.numel() * 8 for b in Bhost))
    d2h = int(out_host.numel() * 8)
    assert np.array_equal(out_host.numpy(), A_dev), "host and device entry points disagree"

    ms, e2e_s = max_over_ranks([ms, e2e_s], world, "cuda")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    ms_step = ms / args.steps
    value = whole_job_value(n_shells, args.steps, world, ms * 1e-3)
    kern_ms = stage[1] / args.steps                                     # the kernel(s) of steps 5-6(iii)
    achieved = (f_con + f_asm) / (kern_ms * 1e-3) / 1e12
    peak_dfma, peak_dmma = sf.sf_fp64_peak(0), sf.sf_fp64_peak(1)
    peak = max(peak_dfma, peak_dmma)
    peak_smem = sf.sf_fp64_peak(2)       # the bare shared-memory-fed MMA loop of the gather-GEMMs (10 LDS.64 per 16 DMMA): context, not the denominator
    peak_source = ("measured in this process: FP64 DFMA %.2f, DMMA(mma.sync m8n8k4) %.2f TFLOP/s; a shared-memory-fed DMMA loop "
                   "reaches %.2f" % (peak_dfma, peak_dmma, peak_smem))
    hbm, hbm_src = hbm_peak()
    # {6j} gathers (step 4): the S arrays, 8 B read from the table + 8 B written per element, over the event time of the stage
    n_s_elems = sf.sf_slice_elems(two_j, two_dl)
    s_ms = stage[0] / args.steps
    sixj_gather = {"elements": n_s_elems, "algorithmic_bytes": 16.0 * n_s_elems, "ms_per_step": s_ms,
                   "achieved": 16.0 * n_s_elems / (s_ms * 1e-3) / 1e9 if s_ms > 0 else None, "peak": hbm, "unit": "GB/s",
                   "bound": "hbm", "peak_source": hbm_src,
                   "note": "random 8-byte reads of the canonical table (32-byte sectors) + dense writes"}
    if sixj_gather["achieved"]:
        sixj_gather["frac"] = sixj_gather["achieved"] / hbm
    if last_path == 4:
        # Factorised path.  Numerator = USEFUL flop per kernel: 2 x the multiply-adds on the index combinations the triangle
        # inequalities allow (host count, no padding).  The executed work (512 flop per issued DMMA.8x8x4, counted by the
        # kernels themselves, padding included) is reported as executed_over_useful, the padding tax.
        flop, mac, elems = factor_work(sf, two_j, two_dl)
        qpk = {4: "k_fz_qp4", 2: "k_fz_qp2", 1: "k_fz_qp"}.get(sf.sf_last_qp_kernel(), "k_fz_qp")
        rk = "k_fz_r2" if args.variant & 1 else "k_fz_gemm<FzMapR>" if args.variant & 8 else "k_fz_r3"
        names = {"qp": qpk + " (Q = sum_l45, P = sum_k4)", "R": rk + " (R = sum_{l34 l35})",
                 "A": "k_fz_gemm<FzMapA> (A' = sum_{k3 x l23})"}
        per = {}
        for k, key in enumerate(("qp", "R", "A")):
            ms_k = kms[k] / args.steps
            tf = flop[key] / (ms_k * 1e-3) / 1e12 if ms_k > 0 else 0.0
            per[key] = {"kernel": names[key], "ms_per_step": ms_k, "useful_flop_per_step": flop[key], "useful_tflops": tf,
                        "frac": tf / peak, "executed_dmma_per_step": dmma[k],
                        "executed_over_useful": 512.0 * dmma[k] / flop[key] if flop[key] > 0 else None,
                        "pipe_busy_frac": 512.0 * dmma[k] / (ms_k * 1e-3) / 1e12 / peak if ms_k > 0 else None}
        dom = max(per, key=lambda n: per[n]["ms_per_step"])
        useful_all = sum(flop.values())
        t_all = sum(kms) / args.steps
        dram = ncu_dram_per_step() if cfg["name"] == wl.CONFIGS[3]["name"] else None
        alg_bytes = 8.0 * 2.0 * (elems["P"] + elems["R"])
        roofline = {"bound": "alu", "kernel": per[dom]["kernel"], "achieved": per[dom]["useful_tflops"], "peak": peak,
                    "unit": "TFLOP/s", "frac": per[dom]["frac"],
                    "traffic": (dram["per_kernel"].get(dom, {}).get("bytes", 0.0) / max(1, dram["per_kernel"].get(dom, {}).get("launches", 1))
                                if dram else None),
                    "traffic_note": "DRAM bytes per launch of the dominant kernel (mean over its launches of one step)",
                    "traffic_source": dram["source"] if dram else None,
                    "traffic_kind": "replayed: read from the committed ncu launch list named in traffic_source, NOT measured in this run" if dram else None,
                    "peak_source": peak_source,
                    "definition": "useful FP64 flop (2 x multiply-adds on valid index ranges, sf_factor_work) / CUDA-event time",
                    "kernels": per,
                    "whole_chain": {"useful_flop_per_step": useful_all, "ms_per_step": t_all,
                                    "useful_tflops": useful_all / (t_all * 1e-3) / 1e12,
                                    "frac": useful_all / (t_all * 1e-3) / 1e12 / peak},
                    "precompute_ms_per_step": kms[3] / args.steps,
                    "hbm": {"algorithmic_bytes_per_step": alg_bytes,
                            "algorithmic_note": "intermediates P and R written once and read once (8 B per structurally non-zero entry); "
                                                "inputs and output are < 0.2 GB",
                            "dram_bytes_per_step": dram["total"] if dram else None,
                            "dram_per_kernel": dram["per_kernel"] if dram else None,
                            "hbm_frac": dram["total"] / (ms_step * 1e-3) / 1e9 / hbm if dram else None,
                            "peak": hbm, "peak_source": hbm_src, "source": dram["source"] if dram else None,
                            "kind": ("replayed: dram_bytes_per_step / dram_per_kernel are read from the committed ncu launch list "
                                     "in `source` (a capture of the same command on the same kernels), not measured in this run; "
                                     "hbm_frac divides them by this run's time") if dram else None}}
    else:
        roofline = {"bound": "alu", "kernel": {3: "k_vertex_line"}.get(last_path, "k_stage_*"),
                    "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "traffic": None,
                    "peak_source": peak_source, "flop_per_step": {"contraction": f_con, "assembly": f_asm},
                    "definition": "SURVEY.md 8(d): F_con + F_asm on valid ranges / CUDA-event time of steps 5-6(iii)",
                    "kernel_ms": kern_ms}
    # the per-shell method of the paper (sf_set_path 3: one {15j} assembly and four mode products per shell) on SURVEY.md 8(d)'s
    # own flop count, timed in this run: 1 warm-up + 2 steps
    per_shell = None
    if last_path == 4 and args.path == 0 and cfg["name"] == wl.CONFIGS[3]["name"] and world == 1 and not args.no_extras:
        try:
            sf.sf_set_path(3)
            sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, stream)
            torch.cuda.synchronize()
            sf.sf_set_timing(True)
            st3 = np.zeros(3)
            for _ in range(2):
                flush.zero_()
                sf.sf_vertex_amplitude(two_j, two_dl, Bdev, out, stream)
                st3 += np.array(sf.sf_last_stage_ms())
            sf.sf_set_timing(False)
            k3 = st3[1] / 2
            tf3 = (f_con + f_asm) / (k3 * 1e-3) / 1e12
            per_shell = {"kernel": "k_vertex_line", "ms_per_step": float(st3.sum() / 2), "kernel_ms": k3,
                         "flop_per_step": {"contraction": f_con, "assembly": f_asm}, "achieved": tf3, "unit": "TFLOP/s",
                         "peak": peak, "frac": tf3 / peak, "shells_per_s": n_shells / (st3.sum() / 2 * 1e-3),
                         "max_abs_diff_vs_factorised_over_max": float(np.abs(out.cpu().numpy() - A_dev).max() / np.abs(A_dev).max()),
                         "definition": "SURVEY.md 8(d): F_con + F_asm on valid ranges / CUDA-event time of steps 5-6(iii)"}
        except sf.SfError as e:
            per_shell = {"unavailable": str(e)}
        finally:
            sf.sf_set_timing(False)
            sf.sf_set_path(args.path)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": cfg["name"], "two_j": two_j, "two_dl": two_dl, "shells": n_shells,
                   "nonempty_shells": work["n_nonempty"], "out_shape": n_i, "boosters": "seeded N(0,1)*(1+u+v+w)^-1.5",
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": "256 MiB device memset between steps (inside the timed region)",
                   "sixj_table_two_jmax": args.table, "path": PATH_NAMES.get(last_path, "?")},
        "vertex_tensors_per_s": world * args.steps / (ms * 1e-3),
        "clocks": clocks,
        "e2e": {"value": whole_job_value(n_shells, args.steps, world, e2e_s), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": 1e3 * e2e_s / args.steps},
        "gpu_launches": launches,
        "value_note": ("shells-equivalent: nominal shells of the tensor / time; the factorised path sums eq. (3) spin by spin and "
                       "never iterates shells (per_shell_path has the per-shell method)" if last_path == 4 else "shells iterated"),
        "roofline": roofline,
        "per_shell_path": per_shell,
        "sixj_gather": sixj_gather,
        "stages_ms_per_step": {"s_arrays": stage[0] / args.steps, "assembly_contraction": kern_ms,
                               "accumulate_normalise": stage[2] / args.steps},
        "sixj_table_build_ms": table_ms,
    }
    if world == 1 and not args.no_extras:
        line["contractions"] = bench_contractions(torch, sf, stream)
        if cfg["name"] == wl.CONFIGS[3]["name"] and args.path == 0:
            line["other_workloads"] = bench_other_workloads(torch, sf, stream, peak)
            line["many_vertices"] = bench_many_vertices(torch, sf, stream)
    if world == 1 and not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        n_sample = min(args.ref_shells, n_shells)
        lo, hi, S = oracle_sample(cfg, B, n_sample)
        dt, r = oracle_time(cfg, B, lo, hi, S, cores)
        line["cpu_baseline"] = {"value": (hi - lo) / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"shells [{lo},{hi}) of {n_shells} (seeded contiguous range, {dt:.1f} s), "
                                          "exact-6j S arrays precomputed untimed"}
        # the same sample through the CUDA path: a parity spot check at the bench's launch configuration
        sub = torch.zeros(tuple(n_i), dtype=torch.float64, device="cuda")
        sf.sf_vertex_amplitude_range(two_j, two_dl, Bdev, lo, hi, sub, stream)
        torch.cuda.synchronize()
        scale = float(np.abs(r["A"]).max())
        line["cpu_baseline"]["max_abs_diff_over_max"] = float(np.abs(sub.cpu().numpy() - r["A"]).max() / scale)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--sub", type=int, default=None, help="Delta_l of config 2")
    ap.add_argument("--table", type=int, default=60, help="two_jmax of the resident {6j} table (-1: none)")
    ap.add_argument("--ref-shells", type=int, default=8000, help="shells in the oracle's bounded sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the secondary rows (other workloads, contractions, per-shell path)")
    ap.add_argument("--one-step-only", action="store_true", help="profiling aid: table build + one vertex call, then exit")
    ap.add_argument("--variant", type=int, default=0, help="kernel variants of the factorised path (sf_set_factor_variant); 0 = default")
    ap.add_argument("--path", type=int, default=0, help="0 automatic (fastest that fits), 1 staged, 3 line, 4 factorised")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = workload(args.config, args.sub)
    if args.impl == "reference":
        run_reference(args, cfg, rank)
    else:
        run_ours(args, cfg, rank, world, local_rank)


if __name__ == "__main__":
    main()
