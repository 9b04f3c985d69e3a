#!/usr/bin/env python
"""bench.py -- throughput of the GBD plane-evaluation hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-cpu-baseline]

Workload: BASELINE.json configs[3] ("C3", the config the metric's roofline fraction is quoted on):
31,757 beamlets x 1024x1024 px, fp64.  One step = the whole hot path on one batch of synthetic
input: gbd_beamlets_create (a1) + gbd_propagate_q (a2) + gbd_eval_field (a3 pre-pass + a4 field sum).
With N > 1 ranks the path is sharded over detector rows with no data-path collective: rank r
evaluates its own 1024-row band of an N-times taller detector (weak scaling).

`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same
workload; it is a deliberately slow program, so the GPU/CPU ratio is context, not a headline.
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
sys.path.insert(0, ROOT)

METRIC = "beamlet-pixel evals/s (fp64)"
UNIT = "evals/s"
WORKLOAD_INDEX = 3
# Roofline bookkeeping of the field-sum kernels, per algorithm (fp64).  `algorithmic` = FP64-pipe instructions per
# (beamlet, pixel) term the evaluation scheme of that kernel needs (DESIGN.md section 6 derives each count).
# `executed`, `traffic` and `other` are NOT typed here: load_capture() reads them at start-up from the ncu summary
# named in `capture` (section `section` of that file), so they cannot drift from the capture of record.  They are what
# ncu measured for that kernel on C3 (thread-level DFMA+DADD+DMUL per term; dram bytes read + written per launch;
# warp instructions per warp-term that are neither FP64-pipe nor F64 conversions) -- not measured in this run, and
# printed with the capture's name.  SURVEY.md 8(d)'s reference count (48, row-hoisted libdevice exp2 + sincospi) is
# reported beside it as `frac_survey_iref48`.
SURVEY_IREF = 48
CAPTURE_TERMS = 31757 * 1024 * 1024          # every capture under profiles/ is one C3 launch (its header says so)
KERNEL_TABLE = {
    # direct: table-driven per-term evaluation on detector-coordinate records with the rounding constants folded into
    # the quadratics (field_fold_kernel): quadratics 4 + h^2 1 + 2^r 3 + tan 2 + cos fold 2 + rotation 2 + accumulate 2
    # = 16 on the FP64 pipe, + 6 / (16 x 8) for the row terms a warp works out once per beamlet (lane l for beamlet l of a
    # group of 16); the two int -> double conversions of the remainders (I2F.F64) run on the XU pipe; the other
    # instructions are 2 x (LOP3 + IMAD + LDS) table lookups, XOR, exponent IMAD, 3/8 slot loads, loops
    "direct": {"kernel": "field_fold_kernel<8,0,0>", "algorithmic": 16 + 6 / (16 * 8), "xu_conversions": 2.0,
               "capture": "profiles/r2_field_fold_kernel_ncu.md", "section": None},
    # recurrence: two direct (polynomial) evaluations per (beamlet, thread) + 10 FP64 instructions per pixel, P = 32
    "recurrence": {"kernel": "field_recur_kernel<32,0,0>", "algorithmic": (65 + 10 * 32) / 32,
                   "capture": "profiles/r2_other_kernels_ncu.md", "section": "## fp64 recurrence"},
    # separable: 4 multiply-adds per pixel + twelve 16-value edge recurrences per 128 x 64 tile
    "separable": {"kernel": "field_sep_kernel<0>", "algorithmic": (4 * 8192 + 12 * (65 + 8 * 16)) / 8192,
                  "capture": "profiles/r2_other_kernels_ncu.md", "section": "## fp64 separable"},
}
_BYTES = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}


def parse_capture(path, section=None):
    """Metric rows (| `name` | unit | value |) of one ncu summary under profiles/: the whole file, or the part from
    the `## ` heading that starts with `section` to the next `## ` heading.  Returns {name: (unit, value)}."""
    rows, inside = {}, section is None
    with open(path) as f:
        for line in f:
            if line.startswith("## "):
                if section is not None:
                    if inside:
                        break
                    inside = line.startswith(section)
                continue
            if not inside or not line.startswith("| `"):
                continue
            cells = [c.strip() for c in line.strip().strip("|").split("|")]
            if len(cells) == 3 and cells[0] not in rows:
                try:
                    rows[cells[0].strip("`")] = (cells[1], float(cells[2]))
                except ValueError:
                    pass
    return rows


def load_capture(kt):
    """Fill executed / traffic / other of a KERNEL_TABLE entry from its ncu summary (None when the file or a row is
    missing: the bench line then says so instead of quoting a remembered number)."""
    kt.update(executed=None, traffic=None, other=None)
    try:
        r = parse_capture(os.path.join(ROOT, kt["capture"]), kt["section"])
        cyc = r["sm__cycles_elapsed.max"][1]
        per_cycle = sum(r[f"smsp__sass_thread_inst_executed_op_{op}_pred_on.sum.per_cycle_elapsed"][1]
                        for op in ("dfma", "dadd", "dmul"))
        kt["executed"] = per_cycle * cyc / CAPTURE_TERMS
        kt["traffic"] = int(round(sum(_BYTES[r[m][0]] * r[m][1] for m in ("dram__bytes_read.sum",
                                                                           "dram__bytes_write.sum"))))
        kt["other"] = (r["smsp__inst_executed.sum"][1] / (CAPTURE_TERMS / 32.0) - kt["executed"]
                       - kt.get("xu_conversions", 0.0))
    except (OSError, KeyError):
        pass
    return kt


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--algo", default="direct", choices=["direct", "recurrence", "separable"],
                    help="field-sum algorithm of the timed path (headline: direct, the per-term evaluation "
                         "BASELINE.json describes; recurrence is reported beside it either way)")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "mixed"],
                    help="fp64 (the headline metric) or mixed (fp64 phase, fp32 envelope / accumulation; BASELINE.json "
                         "configs[3] asks for both); mixed lines report their own pipe roofline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true",
                    help="skip the eval_field_modes / c2_sweep context measurements after the timed region "
                         "(used for the ncu launch list, which then shows the timed step only)")
    ap.add_argument("--cpu-baseline-seconds", type=float, default=12.0)
    return ap.parse_args()


# --------------------------------------------------------------------------- clocks sampler

class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons of one GPU every 200 ms in a thread."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self._stop, self._t = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True,
                                     text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            self._stop.wait(0.2)

    def start(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()

    def stop(self) -> dict:
        self._stop.set()
        if self._t:
            self._t.join(timeout=6)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except Exception:
                continue
            for nm, val in zip(names, r[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "samples": len(sm),
                "reasons": sorted(reasons)}


# --------------------------------------------------------------------------- CPU oracle timing

def oracle_sample(w, seconds: float, threads: int = 0):
    """Time the oracle (a1..a4) on a row sample of workload w sized for ~`seconds` of CPU work, on `threads`
    OpenMP threads (0: all the box exposes).  Returns (evals_per_s, cores, description, elapsed, terms)."""
    import gen
    import oracle
    all_threads = oracle.num_threads()
    if threads:
        oracle.set_num_threads(threads)
    try:
        return _oracle_sample(gen, oracle, w, seconds)
    finally:
        oracle.set_num_threads(all_threads)


def _oracle_sample(gen, oracle, w, seconds):
    cores = oracle.num_threads()
    t0 = time.perf_counter()
    xy0 = oracle.lattice(w.n_across, w.pupil_diameter)
    inp = gen.make_inputs(w, xy0)
    rec = oracle.propagate(inp["xy"], oracle.waist(w.overlap_factor, w.pitch), w.wavelength,
                           inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"], inp["weight"])
    rd = oracle.to_detector(rec, inp["detector"])
    det = inp["detector"]
    n_b = rd.shape[0]
    # probe: `cores` rows, then scale
    t1 = time.perf_counter()
    oracle.field_rows(rd, det, w.wavelength, 0, min(cores, det["n_v"]), 1)
    dt = time.perf_counter() - t1
    per_row = dt / min(cores, det["n_v"])
    n_rows = int(max(cores, min(det["n_v"], seconds / max(per_row, 1e-9))))
    n_rows = max(cores, (n_rows // cores) * cores)
    step = max(1, det["n_v"] // n_rows)
    rows = list(range(0, det["n_v"], step))[:n_rows]
    t2 = time.perf_counter()
    oracle.field_rows(rd, det, w.wavelength, 0, rows[-1] + 1, step)
    el = time.perf_counter() - t2
    terms = len(rows) * det["n_u"] * n_b
    desc = (f"{len(rows)} of {det['n_v']} detector rows (every {step}th from row 0) x {det['n_u']} px "
            f"x {n_b} beamlets of {w.name}; OpenMP over rows")
    return terms / el, cores, desc, el, terms


def run_reference(args):
    """--impl reference: the oracle, as it stands, on host cores; bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import gen
    import oracle
    w = gen.workload(WORKLOAD_INDEX)
    cores = oracle.num_threads()
    xy0 = oracle.lattice(w.n_across, w.pupil_diameter)
    inp = gen.make_inputs(w, xy0)
    det = inp["detector"]
    n_rows = cores                                  # one row per thread per step
    step_rows = max(1, det["n_v"] // n_rows)
    times = []
    terms = 0
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        xy = oracle.lattice(w.n_across, w.pupil_diameter)
        rec = oracle.propagate(inp["xy"], oracle.waist(w.overlap_factor, w.pitch), w.wavelength,
                               inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"], inp["weight"])
        rd = oracle.to_detector(rec, det)
        oracle.field_rows(rd, det, w.wavelength, 0, (n_rows - 1) * step_rows + 1, step_rows)
        dt = time.perf_counter() - t0
        terms = n_rows * det["n_u"] * rd.shape[0]
        if i >= args.warmup:
            times.append(dt)
        del xy
    ms = 1e3 * sum(times) / len(times)
    value = terms / (ms * 1e-3)
    sample = (f"each step: a1+a2+a3 in full and the field sum on {n_rows} of {det['n_v']} rows "
              f"(every {step_rows}th) x {det['n_u']} px x {w.n_across}-across lattice of {w.name}")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "C3 large-focal-plane (BASELINE.json configs[3]), bounded sample",
                       "beamlets": int(terms // (n_rows * det["n_u"])), "detector": [det["n_v"], det["n_u"]]},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------- per-config table

def config_table(G, gen, dev, reps=5):
    """For C0..C5: device milliseconds of gbd_beamlets_create + gbd_propagate_q + gbd_eval_field (CUDA events, best of
    `reps`, inputs resident; C5 also times gbd_trace_mirrors, which derives its ABCD), evals/s, and the field against
    the CPU oracle -- every pixel where the oracle needs under a second, else every (n_v / 16)-th row: relative L2
    and the worst pixel relative to the peak.  C3 also in mixed precision (BASELINE.json configs[3]: "in both").
    The oracle is used here the way cpu_baseline uses it: as the reported checker, outside every timed region."""
    import numpy as np
    import torch
    import oracle
    rows_out = []
    for idx, precision in ((0, 0), (1, 0), (2, 0), (3, 0), (3, 1), (4, 0), (5, 0)):
        w = gen.workload(idx)
        g = G.run_workload(w, gen.make_inputs, precision=precision, device=dev)      # untimed: inputs + the field to check
        b, inp = g["beamlets"], g["inputs"]
        det = inp["detector"]
        terms = b.n * det["n_u"] * det["n_v"]
        d_in = {k: (None if inp[k] is None else torch.as_tensor(inp[k], device=dev)) for k in ("abcd", "base", "weight")}
        params, field = g["params"], g["field"]
        ws = torch.empty(G.eval_workspace_bytes(b, det, precision), dtype=torch.uint8, device=dev)
        spec = inp.get("trace")

        def path():
            bb = G.beamlets_create(w.n_across, w.pupil_diameter, w.overlap_factor, w.wavelength, device=dev)
            if spec is not None:
                G.trace_mirrors(bb, spec, spec.get("p_in"), spec.get("opl0"))
            G.propagate_q(b, inp["abcd_mode"], d_in["abcd"], inp["l0"], d_in["base"], d_in["weight"], out=params)
            G.eval_field(b, det, precision=precision, out=field, workspace=ws)

        path()
        torch.cuda.synchronize()
        best = float("inf")
        for _ in range(reps):
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record()
            path()
            a1.record()
            torch.cuda.synchronize()
            best = min(best, a0.elapsed_time(a1))
        step = 1 if terms <= 6e8 else max(1, det["n_v"] // 16)
        ref = oracle.run_workload(w, gen.make_inputs, rows=None if step == 1 else (0, det["n_v"], step))["field"][::step]
        got = field.cpu().numpy()[::step].astype(np.complex128)
        rows_out.append({"config": w.name, "precision": "mixed" if precision else "fp64", "beamlets": b.n,
                         "detector": [det["n_v"], det["n_u"]], "terms": terms, "ms": best,
                         "evals_per_s": terms / (best * 1e-3),
                         "rel_l2_vs_oracle": float(np.linalg.norm(got - ref) / np.linalg.norm(ref)),
                         "worst_pixel_vs_peak": float(np.max(np.abs(got - ref)) / np.max(np.abs(ref))),
                         "oracle_rows": "all" if step == 1 else f"every {step}th of {det['n_v']}"})
    return rows_out


# --------------------------------------------------------------------------- strong scaling (N > 1)

def strong_scaling(evaluate, detector, rank, world, dist, steps, device=None, flush=None):
    """SURVEY.md 8(e) as it is written: ONE detector whose rows are partitioned across the ranks
    (sharding.row_band; every rank holds all beamlet records, no collective on the data path), then the one optional
    collective after the path, the all-gather of the finished bands (sharding.gather_rows, 16 B per pixel), timed
    separately.  `evaluate(band_detector)` returns this rank's (rows, n_u) complex tensor with the work enqueued on
    the current stream (device tensors) or done (host tensors: the gloo CPU test drives this function with the oracle
    as evaluator).  Times are device times (CUDA events) for device tensors, MAX over ranks, per step.
    Returns (summary dict, the gathered (n_v, n_u) field of the last step)."""
    import torch
    from paper_2404_12454_b200 import sharding
    on_gpu = device is not None and torch.device(device).type == "cuda"

    def sync():
        if on_gpu:
            torch.cuda.synchronize()

    def timed(fn):
        """(result, milliseconds) of fn(): CUDA events on the current stream, or the host clock for host tensors."""
        if on_gpu:
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            out = fn()
            b.record()
            torch.cuda.synchronize()
            return out, a.elapsed_time(b)
        t0 = time.perf_counter()
        out = fn()
        return out, 1e3 * (time.perf_counter() - t0)

    n_v = int(detector["n_v"])
    band = sharding.row_band(detector, rank, world)
    full = sharding.gather_rows(evaluate(band), n_v)            # warm-up of both (NCCL opens its channels here)
    sync()
    eval_ms = gather_ms = 0.0
    for _ in range(steps):
        if flush is not None:
            flush()
        sync()
        dist.barrier()
        mine, ms = timed(lambda: evaluate(band))
        eval_ms += ms
        dist.barrier()
        full, ms = timed(lambda: sharding.gather_rows(mine, n_v))
        gather_ms += ms
    t = torch.tensor([eval_ms, gather_ms], dtype=torch.float64, device=device if on_gpu else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    rows = [sharding.row_range(n_v, r, world) for r in range(world)]
    return {"scaling": "strong", "what": "ONE detector, rows partitioned across the ranks (sharding.row_band), no "
                                         "collective on the data path; then sharding.gather_rows (all-gather of "
                                         "the finished bands), timed separately; max over ranks",
            "world": world, "rows_per_rank": [b - a for a, b in rows], "steps": steps,
            "eval_ms_per_step": float(t[0]) / steps, "gather_ms_per_step": float(t[1]) / steps,
            "gather_bytes_per_rank": int(full.numel() * full.element_size())}, full


# --------------------------------------------------------------------------- our arm

def run_ours(args):
    import numpy as np
    import torch
    import gen
    import paper_2404_12454_b200 as G

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit(f"bench.py: rank {rank} of {world}: no CUDA device (there is no CPU fallback; use --impl "
                         "reference for the CPU oracle)")
    if local >= torch.cuda.device_count():
        raise SystemExit(f"bench.py: rank {rank} of {world}: local rank {local} but only "
                         f"{torch.cuda.device_count()} CUDA device(s) are visible")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    G.load_library()

    w = gen.workload(WORKLOAD_INDEX)
    K, W = args.steps, max(args.warmup, 3)

    # ---- setup (untimed): seeded inputs; rank r gets its own band of an N-times taller detector
    b0 = G.beamlets_create(w.n_across, w.pupil_diameter, w.overlap_factor, w.wavelength, device=dev)
    inp = gen.make_inputs(w, b0.positions.cpu().numpy())
    from paper_2404_12454_b200 import sharding
    det = sharding.weak_band(inp["detector"], rank, world)
    n_b = b0.n
    n_px = det["n_u"] * det["n_v"]
    terms = n_b * n_px
    d_abcd = torch.as_tensor(inp["abcd"], device=dev)
    d_weight = torch.as_tensor(inp["weight"], device=dev)
    mixed = args.precision == "mixed"
    prec = G.PRECISION_MIXED if mixed else G.PRECISION_FP64
    cdtype = torch.complex64 if mixed else torch.complex128
    field = torch.empty((det["n_v"], det["n_u"]), dtype=cdtype, device=dev)
    params = torch.empty((n_b, G.gbd.NREC), dtype=torch.float64, device=dev)
    ws = torch.empty(G.eval_workspace_bytes(b0, det), dtype=torch.uint8, device=dev)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)     # > 126 MB L2
    ev_k0 = torch.cuda.Event(enable_timing=True)
    ev_k1 = torch.cuda.Event(enable_timing=True)

    algo = {"direct": G.ALGO_DIRECT, "recurrence": G.ALGO_RECURRENCE, "separable": G.ALGO_SEPARABLE}[args.algo]
    # algorithmic FP64-pipe instructions per term of the timed kernel
    kt = load_capture(KERNEL_TABLE[args.algo])
    instr_per_term = kt["algorithmic"]

    def step():
        """The whole hot path, inputs resident in HBM."""
        b = G.beamlets_create(w.n_across, w.pupil_diameter, w.overlap_factor, w.wavelength, device=dev)
        G.propagate_q(b, inp["abcd_mode"], d_abcd, inp["l0"], None, d_weight, out=params)
        G.eval_field(b, det, out=field, workspace=ws, algo=algo, precision=prec)
        return b

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(W):
        step()
        flush.zero_()
    # ---- FP64 peak probe (roofline denominator), burst
    G.probe_dfma(2000, device=dev)
    torch.cuda.synchronize()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    n_dfma = G.probe_dfma(20000, device=dev)
    p1.record()
    torch.cuda.synchronize()
    dfma_rate = n_dfma / (p0.elapsed_time(p1) * 1e-3)

    # ---- timed region: exactly K steps; device time per step by CUDA events, L2 flushed between
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    launches0 = G.launch_count()
    G.set_profile_events(ev_k0, ev_k1)
    step_ms, kern_ms = [], []
    t_wall0 = time.perf_counter()
    for _ in range(K):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        step()
        e1.record()
        torch.cuda.synchronize()
        step_ms.append(e0.elapsed_time(e1))
        kern_ms.append(ev_k0.elapsed_time(ev_k1))
        flush.zero_()
    barrier()
    t_wall = time.perf_counter() - t_wall0
    G.set_profile_events(None, None)
    launches = G.launch_count() - launches0
    clocks = sampler.stop()
    sampler_clock_mhz = clocks.get("sm_mhz")
    total_ms = sum(step_ms)
    if dist is not None:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms_per_step = total_ms / K
    value = world * terms / (ms_per_step * 1e-3)

    # ---- end to end through the C ABI with HOST buffers (pinned), H2D + D2H inside the timed region
    h_xy = torch.as_tensor(inp["xy"]).contiguous().pin_memory()
    h_abcd = torch.as_tensor(inp["abcd"]).contiguous().pin_memory()
    h_weight = torch.as_tensor(inp["weight"]).contiguous().pin_memory()
    h_field = torch.empty((det["n_v"], det["n_u"]), dtype=cdtype).pin_memory()
    hws = torch.empty(G.host_workspace_bytes(b0, det, inp["abcd_mode"]), dtype=torch.uint8, device=dev)

    def e2e_step():
        G.eval_field_host(b0, h_xy, inp["abcd_mode"], h_abcd, inp["l0"], None, h_weight, det,
                          h_field, hws, algo=algo, precision=prec)

    for _ in range(2):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(K):
        e2e_step()                                   # synchronises the stream itself
    barrier()
    e2e_s = time.perf_counter() - t0
    if dist is not None:
        t = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    e2e_value = world * terms * K / e2e_s
    h2d = (h_xy.numel() + h_abcd.numel() + h_weight.numel()) * 8
    d2h = h_field.numel() * h_field.element_size()
    checksum = float(h_field.abs().sum().item())

    # ---- N > 1: SURVEY 8(e)'s partition of ONE C3 detector across the ranks + the all-gather of the bands
    strong = None
    if dist is not None:
        full_det = inp["detector"]
        band_rows = -(-int(full_det["n_v"]) // world)
        band_field = torch.empty((band_rows, full_det["n_u"]), dtype=cdtype, device=dev)

        def eval_band(band):
            return G.eval_field(b0, band, params=params, out=band_field[: band["n_v"]], workspace=ws, algo=algo,
                                precision=prec)

        strong, full_field = strong_scaling(eval_band, full_det, rank, world, dist, K, device=dev,
                                            flush=flush.zero_)
        full_terms = n_b * int(full_det["n_u"]) * int(full_det["n_v"])
        strong.update(value=full_terms / (strong["eval_ms_per_step"] * 1e-3), unit=UNIT,
                      value_with_gather=full_terms / ((strong["eval_ms_per_step"] + strong["gather_ms_per_step"])
                                                      * 1e-3),
                      backend=dist.get_backend(), nccl_world=dist.get_world_size(),
                      checksum_abs_sum=float(full_field.abs().sum().item()))
        del full_field

    # ---- the other modes of the same field sum (gbd_eval_field only, device time), for context
    def time_eval(**kw):
        out = G.eval_field(b0, det, params=params, workspace=ws, **kw)
        torch.cuda.synchronize()
        ts = []
        for _ in range(5):
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record()
            G.eval_field(b0, det, params=params, out=out, workspace=ws, **kw)
            a1.record()
            torch.cuda.synchronize()
            ts.append(a0.elapsed_time(a1))
        ms = sum(ts) / len(ts)
        return {"ms": ms, "evals_per_s": terms / (ms * 1e-3)}
    other_modes = None if args.no_extras else {
                   "fp64_direct": time_eval(algo=G.ALGO_DIRECT),
                   "fp64_recurrence": time_eval(algo=G.ALGO_RECURRENCE),
                   "fp64_separable": time_eval(algo=G.ALGO_SEPARABLE),
                   "mixed_direct": time_eval(precision=G.PRECISION_MIXED),
                   "mixed_recurrence": time_eval(precision=G.PRECISION_MIXED, algo=G.ALGO_RECURRENCE),
                   "mixed_separable": time_eval(precision=G.PRECISION_MIXED, algo=G.ALGO_SEPARABLE)}

    # ---- Hermite-Gaussian beamlets (orders <= 2) on the same workload: gbd_eval_field_modes, for context
    if other_modes is not None:
        rng = np.random.default_rng(7)
        mw = torch.as_tensor(rng.standard_normal((12, n_b)), device=dev)
        modes = G.hg_modes(b0, inp["abcd_mode"], d_abcd, mw)
        wsm = torch.empty(G.load_library().gbd_eval_modes_workspace_bytes(b0._h, G.gbd.C.byref(G.Detector.from_dict(det))),
                          dtype=torch.uint8, device=dev)
        outm = G.eval_field_modes(b0, modes, det, params=params, workspace=wsm)
        torch.cuda.synchronize()
        ts = []
        for _ in range(5):
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record()
            G.eval_field_modes(b0, modes, det, params=params, out=outm, workspace=wsm)
            a1.record()
            torch.cuda.synchronize()
            ts.append(a0.elapsed_time(a1))
        other_modes["fp64_direct_hermite_gaussian_modes"] = {"ms": sum(ts) / len(ts),
                                                              "evals_per_s": terms / (sum(ts) / len(ts) * 1e-3)}

    # ---- the paper's beamlet-parameter search (C2: 90 runs) through gbd_airy_sweep, for context
    sweep = None
    if world == 1 and not args.no_extras:
        ws_runs = gen.sweep_workloads()
        w2 = ws_runs[0]
        det2 = gen.detector_dict(w2)
        runs = [(x.n_across, x.pupil_diameter, x.overlap_factor, x.wavelength) for x in ws_runs]
        abcd2 = torch.as_tensor(gen.ideal_lens_abcd(w2.focal_length).reshape(16), device=dev)
        terms2 = sum(G.lattice_count(x.n_across, x.pupil_diameter) for x in ws_runs) * det2["n_u"] * det2["n_v"]
        sweep = {"runs": len(runs), "terms": terms2,
                 "what": "gbd_airy_sweep: lattice + parameters + field + Airy RMS metrics of all runs, "
                         "wall time of the call plus the read-back of the [90][10] result"}
        for nm, al in (("direct", G.ALGO_DIRECT), ("recurrence", G.ALGO_RECURRENCE),
                       ("separable", G.ALGO_SEPARABLE)):
            best = None
            for _ in range(4):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                res = G.airy_sweep(runs, abcd2, w2.focal_length, det2, w2.wavelength * w2.f_number,
                                   algo=al, device=dev).cpu()
                dt = time.perf_counter() - t0
                best = dt if best is None else min(best, dt)
            sweep[nm] = {"ms": best * 1e3, "evals_per_s": terms2 / best,
                         "rms_vs_airy_N51_OF3": float(res[44, 0])}

    # ---- the point-evaluation baseline against the plane evaluation on the shape of the paper's runtime experiment
    #      (Fig. 7: one 256 x 256 px PSF against the number of beamlets across the pupil), for context
    point_eval = None
    if world == 1 and not args.no_extras:
        def best_ms(fn, reps=3):
            fn()
            torch.cuda.synchronize()
            best = None
            for _ in range(reps):
                a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a0.record()
                fn()
                a1.record()
                torch.cuda.synchronize()
                best = a0.elapsed_time(a1) if best is None else min(best, a0.elapsed_time(a1))
            return best
        rows = []
        for n_ac in (11, 31, 51, 71, 101):
            wp = gen.workload(2, n_ac, 1.5)
            gp = G.run_workload(wp, gen.make_inputs, device=dev)
            bp, ip = gp["beamlets"], gp["inputs"]
            ab = torch.as_tensor(ip["abcd"], device=dev)
            pe = best_ms(lambda: G.eval_field_pointwise(bp, 1, ab, ip["l0"], None, None, ip["detector"]))
            pl = {nm: best_ms(lambda al=al: G.eval_field(bp, ip["detector"], algo=al, workspace=bp._ws))
                  for nm, al in (("direct", G.ALGO_DIRECT), ("recurrence", G.ALGO_RECURRENCE),
                                 ("separable", G.ALGO_SEPARABLE))}
            rows.append({"beamlets_across": n_ac, "beamlets": bp.n, "point_ms": pe, "plane_ms": pl,
                         "point_over_plane_direct": pe / pl["direct"],
                         "point_over_plane_best": pe / min(pl.values())})
        point_eval = {"what": "gbd_eval_field_pointwise (P:88-100 steps 2-5 per pixel and beamlet) against gbd_eval_field "
                              "on 256 x 256 px, ideal f/3.9 lens (C2 optics); device time of the call, best of 3",
                      "paper": "P:233 Fig. 7: plane / point 34x on its CPU; on its GPU (V100S, cupy array code) point "
                               "evaluation runs 39x and plane evaluation 1,760x faster than on the CPU; GPU plane "
                               "against CPU point 67,513x, hence plane / point on the GPU about 67,513 / 39 = 1,731x",
                      "rows": rows}

    # ---- (5) the paper's Fig. 5 experiment on the HST-like telescope of Table 2 (workload C5, rays traced by
    #      gbd_trace_mirrors): both algorithms against the Airy pattern, and their run times
    hst_psf = None
    if world == 1 and not args.no_extras:
        w5 = gen.workload(5)
        g5 = G.run_workload(w5, gen.make_inputs, device=dev)
        b5, i5 = g5["beamlets"], g5["inputs"]
        det5 = i5["detector"]
        det1 = dict(det5, n_u=1, n_v=1)
        lfn = w5.wavelength * w5.f_number
        pw_args = (b5, i5["abcd_mode"], i5["abcd"], i5["l0"], i5["base"], i5["weight"])
        plane_ms = best_ms(lambda: G.eval_field(b5, det5, workspace=b5._ws))
        point_ms = best_ms(lambda: G.eval_field_pointwise(*pw_args, det5))
        m_plane = G.psf_metrics(G.eval_field(b5, det5), det5, lfn, G.eval_field(b5, det1)).cpu().numpy()
        m_point = G.psf_metrics(G.eval_field_pointwise(*pw_args, det5), det5, lfn,
                                G.eval_field_pointwise(*pw_args, det1)).cpu().numpy()
        hst_psf = {"what": "unobscured HST-like Ritchey-Chretien telescope (P:324-327 Table 2; 551 nm, EPD 2.4 m, 512 x 512 px "
                           "of 2.8 mas), 8,021 beamlets traced on the device: peak-normalised PSF against the Airy pattern "
                           "(RMS over the detector) and device time of the field call, best of 3",
                   "paper": "P:202-204 Fig. 5: plane evaluation 113.78 s, point evaluation 1309.11 s (11.5x, one 3 GHz CPU); "
                            "plane-evaluation RMS about half the point-evaluation RMS",
                   "plane": {"ms": plane_ms, "rms_vs_airy": float(m_plane[0]), "max_abs_diff": float(m_plane[8])},
                   "point": {"ms": point_ms, "rms_vs_airy": float(m_point[0]), "max_abs_diff": float(m_point[8])},
                   "point_over_plane_time": point_ms / plane_ms}

    # ---- roofline of the dominant kernel (field sum), this rank
    k_ms = sum(kern_ms) / len(kern_ms)
    achieved = terms * 2 * instr_per_term / (k_ms * 1e-3) / 1e12
    peak = 2.0 * dfma_rate / 1e12
    roofline = {"bound": "alu", "kernel": kt["kernel"],
                "achieved": achieved, "peak": peak,
                "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": kt["traffic"],
                "kernel_ms": k_ms, "kernel_share_of_step": k_ms / (sum(step_ms) / K),
                "algorithmic_fp64_instr_per_term": instr_per_term,
                "frac_pipe": (terms * kt["executed"] / (k_ms * 1e-3) / dfma_rate) if kt["executed"] else None,
                "frac_survey_iref48": terms * SURVEY_IREF / (k_ms * 1e-3) / dfma_rate,
                "from_capture": {"file": kt["capture"], "executed_fp64_instr_per_term": kt["executed"],
                                 "dram_bytes_per_launch": kt["traffic"],
                                 "note": "ncu values of the named capture (C3, fp64), not measured in this run"},
                "peak_source": "FP64-pipe DFMA rate measured in this run by gbd_probe_dfma (8 chains/"
                               "thread, 148*8 CTAs x 256 thr), x2 flop; MEASURED_PEAKS.json has no FP64 "
                               "entry",
                "dfma_per_s": dfma_rate}

    if kt.get("xu_conversions") and kt["other"] is not None and not mixed:
        # The fast direct kernel is bound by the dispatch port of the SM sub-partitions, not by one pipe: a warp
        # instruction of the half-rate FP64 pipe (16 lanes per sub-partition) or an F64 conversion holds the port for 2
        # cycles, every other instruction for 1, and they do not overlap (issue model fitted in round 1).
        clk = 1e6 * (sampler_clock_mhz if sampler_clock_mhz else 1965.0)
        slots = 2.0 * kt["algorithmic"] + 2.0 * kt["xu_conversions"] + kt["other"]
        roofline["dispatch"] = {
            "kind": "issue MODEL fitted to the probes of profiles/r1_fp64_pipe_probes.md -- not a hardware counter",
            "model": "2 dispatch cycles per FP64-pipe or F64-conversion warp instruction, 1 per other instruction",
            "fp64_pipe_instr_per_term": kt["algorithmic"], "xu_f64_conversions_per_term": kt["xu_conversions"],
            "other_instr_per_term": kt["other"], "dispatch_cycles_per_warp_term": slots,
            "measured_cycles_per_warp_term": k_ms * 1e-3 * clk * 148 * 4 / (terms / 32.0),
            "frac": slots * (terms / 32.0) / (k_ms * 1e-3 * clk * 148 * 4),
            "peak_source": f"148 SMs x 4 sub-partitions x {clk / 1e6:.0f} MHz (SM clock sampled during the timed region)"}

    if mixed:
        # mixed precision: the pipe that bounds each algorithm, peak = guide unit count x SM clock under this load
        clk = 1e6 * (sampler_clock_mhz if sampler_clock_mhz else 1965.0)
        if args.algo == "direct":
            # field_mixed_tab_kernel: 18.0 warp instructions per term (SASS of the inner loop: 144 per beamlet and 8
            # pixels -- 2.4 DFMA, 1 MUFU.EX2, 1.6 LDS, 3 integer, 1 I2FP, 8.5 fp32, loop), of which the 2.4 FP64-pipe
            # ones hold the dispatch port for 2 cycles: 20.4 dispatch cycles per warp-term; bound = that port (the XU
            # pipe, which bounded the 3-MUFU kernel this one replaced at 25.7 ms, is at 1 MUFU per term now)
            per, pipe, lanes, kname = 20.4, "dispatch port (1 warp instruction per sub-partition cycle, FP64 2)", 128, \
                "field_mixed_tab_kernel<8,0>"
        elif args.algo == "recurrence":  # 10 FP32 instructions per pixel + two MUFU-path start values per 32 pixels
            per, pipe, lanes, kname = 10.0 + 2 * 20.0 / 32, "fp32 (FFMA/FMUL/FADD)", 128, "field_recur_kernel<32,0,1>"
        else:                            # 4 FFMA per term + sixteen 16-value edge runs per 128 x 128 tile
            per, pipe, lanes, kname = (4 * 16384 + 16 * (40 + 8 * 16)) / 16384, "fp32 (FFMA)", 128, \
                "field_sep_kernel<float,0>"
        peak_i = 148 * lanes * clk
        ach_i = terms * per / (k_ms * 1e-3)
        roofline = {"bound": "alu", "pipe": pipe, "kernel": kname,
                    "achieved": ach_i / 1e12, "peak": peak_i / 1e12, "unit": "Tinstr/s (thread-level)",
                    "frac": ach_i / peak_i, "traffic": None, "kernel_ms": k_ms,
                    "kernel_share_of_step": k_ms / (sum(step_ms) / K),
                    "algorithmic_instr_per_term": per,
                    "peak_source": f"148 SMs x {lanes} lanes x {clk / 1e6:.0f} MHz (B200_PROFILING guide unit "
                                   "counts x the SM clock sampled during the timed region)"}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    # ---- BASELINE.md section 3's table in one place: every BASELINE.json config (and NEXT-1's C5) through the whole
    #      path a1..a4 -- device time of the three calls, and the field against the oracle on a documented row sample
    configs = None
    if not args.no_extras and not args.no_cpu_baseline and world == 1:
        configs = config_table(G, gen, dev)

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        v, cores, desc, el, _ = oracle_sample(w, args.cpu_baseline_seconds)
        v1, _, desc1, el1, _ = oracle_sample(w, args.cpu_baseline_seconds / 3, threads=1)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
               "seconds": el,
               "single_thread": {"value": v1, "unit": UNIT, "cores": 1, "sample": desc1, "seconds": el1}}
    line = {"metric": METRIC if not mixed else "beamlet-pixel evals/s (mixed: fp64 phase, fp32 envelope/accumulation)",
            "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64" if not mixed else "f64 phase + f32", "data": "synthetic",
            "config": {"workload": "C3 large-focal-plane (BASELINE.json configs[3]): f/4 ideal lens, "
                                   "201 beamlets across, OF 2.0, seeded Gaussian-apodised random weights",
                       "beamlets": n_b, "detector": [det["n_v"], det["n_u"]],
                       "terms_per_step_per_gpu": terms, "precision": args.precision, "algo": args.algo,
                       "step": "gbd_beamlets_create + gbd_propagate_q + gbd_eval_field",
                       "sharding": "rank r evaluates its own 1024-row band (no collective)",
                       "l2": "256 MiB buffer written between timed steps (inputs are 3 MB)"},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "call": "gbd_eval_field_host (pinned host buffers)",
                    "checksum_abs_sum": checksum},
            "gpu_launches": launches, "wall_s_timed_region": t_wall, "strong": strong,
            "roofline": roofline, "cpu_baseline": cpu, "configs": configs, "eval_field_modes": other_modes, "c2_sweep": sweep,
            "point_eval": point_eval, "hst_psf": hst_psf}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def respawn_under_torchrun(args) -> int:
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: launch the N ranks ourselves, the way
    the driver does (one process per GPU, rendezvous on 127.0.0.1), and pass their output through.  Rank 0 prints
    the JSON line with n_gpus = N."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    print(f"bench.py: --gpus {args.gpus} without WORLD_SIZE: spawning {args.gpus} ranks: {' '.join(cmd)}",
          file=sys.stderr, flush=True)
    return subprocess.run(cmd).returncode


def main():
    args = parse_args()
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    if args.impl == "reference":
        run_reference(args)
        return
    world = os.environ.get("WORLD_SIZE")
    if world is None and args.gpus > 1:
        sys.exit(respawn_under_torchrun(args))
    if world is not None and int(world) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch one rank per GPU")
    run_ours(args)


if __name__ == "__main__":
    main()
