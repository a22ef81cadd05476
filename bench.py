#!/usr/bin/env python
"""bench.py -- throughput of the PGD hot path on BASELINE.json's workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl reference]

Without --config the run times configs[1], [2], [3] and [4] of BASELINE.json one after the other in one process: the
top-level line is the largest of them (configs[4], named in config.workload) and `per_config` carries value, e2e,
roofline, cpu_baseline, ms_per_step and clocks of each.  --config I times that one configuration alone.

A bench "step" is ONE afs_pgd_run call: the whole hot path (S1..S10 of DESIGN.md) over one batch of B restarts for
the configuration's PGD iteration count.  metric = PGD restart-steps per second = B * pgd_iterations / time.
`value` is measured with X0 already resident in HBM (CUDA events on the launching stream, max over ranks);
`e2e` is the same metric through afs_pgd_run_host: pinned HOST buffers, H2D and D2H copies inside the timed region.
One JSON line is printed by rank 0.  N > 1 (torchrun): every rank runs the full configuration on its own draw of
start points (weak scaling, restarts are independent: PAPER.md L164), no collective inside the loop, one all-gather
of the best counts at the end.
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

import workloads as W  # noqa: E402


# --------------------------------------------------------------------------------------------- algorithmic work
def kernel_class_of_constraints(inst):
    """The library's execution classes (afs_internal.h), restated so that algorithmic work can be attributed to the
    kernel that does it: names are Problem.KERNEL_CLASSES ('var' holds the pull clauses; 'long' is the group of
    launches that serve the LONG class in one iteration: long_scan, long1/3/5/9 by pmf size, glong)."""
    L = inst.lengths()
    ty = inst.types
    prod = (ty == W.AFS_OR) | (ty == W.AFS_XOR)
    two = (ty == W.AFS_NAE) | (ty == W.AFS_EO) | (ty == W.AFS_AMO)
    cnt = (ty == W.AFS_EK) | (ty == W.AFS_CARD)
    out = np.empty(inst.m, dtype=object)
    for c in range(inst.m):
        l = int(L[c])
        if (prod[c] or ty[c] == W.AFS_NAE) and l <= 5:
            out[c] = "var"
        elif prod[c] or two[c]:
            out[c] = "med0"
        elif cnt[c] and l <= 64:
            out[c] = "cmed"
        else:
            out[c] = "long"
    return out


def algorithmic_flops_per_constraint(inst) -> np.ndarray:
    """SURVEY.md 8(d) / DESIGN.md section 7: minimal flops of objective + gradient + chain rule per constraint and
    restart (FMA = 2).  EK / CARD: 6 L K with K = min(k, L-k+1)+1 cells; literals of variables fixed by the mask are
    constants of the run and are folded (L counts the free literals, k is reduced by the fixed true ones)."""
    L = inst.lengths().astype(np.float64)
    k = inst.k.astype(np.float64)
    ty = inst.types
    f = np.zeros_like(L)
    f[ty == W.AFS_OR] = 5 * L[ty == W.AFS_OR] + 2
    f[ty == W.AFS_XOR] = 3 * L[ty == W.AFS_XOR] + 1
    f[ty == W.AFS_NAE] = 9 * L[ty == W.AFS_NAE]
    two = (ty == W.AFS_EO) | (ty == W.AFS_AMO)
    f[two] = 15 * L[two]
    cnt = np.flatnonzero((ty == W.AFS_EK) | (ty == W.AFS_CARD))
    for c in cnt:
        lits = inst.lits[inst.row_ptr[c]:inst.row_ptr[c + 1]]
        Lc, kc = float(len(lits)), float(inst.k[c])
        if inst.mask is not None:
            mv = inst.mask[np.abs(lits) - 1].astype(np.int64)
            fixed = mv != 0
            true_fixed = np.sum(fixed & ((mv < 0) != (lits < 0)))      # literal true: variable True (-1) XOR negated
            Lc -= float(fixed.sum())
            kc -= float(true_fixed)
        K = min(kc, Lc - kc + 1) + 1
        f[c] = 6 * Lc * max(K, 1) if (Lc > 0 and 0 < kc <= Lc) else 0.0
    return f


def algorithmic_work(inst, B=None):
    """Per kernel class and per PGD iteration over B restarts (default: the whole batch): (flops, compulsory HBM bytes).
    The rule of the bench line: a restart's work counts in the iterations in which the method has to move it -- retired
    restarts (fixed points of the PGD map) need none -- so B is the MEAN NUMBER OF ACTIVE restarts per
    iteration for the timed call, and the full batch for the pass timed with retirement switched off."""
    cls = kernel_class_of_constraints(inst)
    f = algorithmic_flops_per_constraint(inst)
    L = inst.lengths().astype(np.float64)
    if inst.mask is not None:      # literals of fixed variables are constants of the run: neither gathered nor written
        fixed = (inst.mask[np.abs(inst.lits) - 1] != 0).astype(np.float64)
        L = L - np.add.reduceat(fixed, inst.row_ptr[:-1]) if inst.m else L
    B = float(inst.B if B is None else B)
    work = {}
    for name in set(cls):
        sel = cls == name
        if name == "var":
            continue
        # compulsory HBM bytes of a materialising kernel: every X element its literals touch once (at most the whole
        # iterate) + its literal CSR.  Per-literal gradient rows are scratch traffic the design has to avoid
        # (SURVEY.md 8(d)), not algorithmic bytes.
        work[name] = (float(f[sel].sum()) * B, min(float(L[sel].sum()), float(inst.n)) * B * 4 + float(L[sel].sum()) * 8)
    pull = cls == "var"
    pushed = float(L[~pull].sum())
    # variable pass: pull clauses, one add per materialised literal gradient, 5 flops per variable for S7-S9;
    # bytes: read X + write X, the materialised gradients once, the pull streams once
    work["var"] = ((float(f[pull].sum()) + pushed + 5.0 * inst.n) * B,
                   2 * B * inst.n * 4 + pushed * B * 4 + float(L[pull].sum() * 4 * 4))
    work["sat_pull"] = (0.0, float(inst.n * B / 8 + L[pull].sum() * 4))
    total_f = float(f.sum() + inst.nnz + 5 * inst.n) * B
    work["step"] = (total_f, float(2 * B * inst.n * 4 + inst.nnz * 4))
    return work


def active_trace(P, X0, pgd_steps, lr, mask, every):
    """Active restarts in each PGD iteration of the timed call, re-derived through the public API (untimed): the call
    retires, after every `every`-th iteration, the restarts whose last step left the iterate unchanged.  The same
    iterates are produced here in chunks without retirement (the PGD map is deterministic, so resuming from X is exact)
    and compared step against step."""
    import torch
    B = X0.shape[0]
    if every <= 0:
        return np.full(pgd_steps, B, dtype=np.int64)
    P.set_option(2, 0)
    X = X0.clone()
    active = torch.ones(B, dtype=torch.bool, device=X.device)
    n_act, t = [], 0
    while t < pgd_steps:
        nxt = min((t // every + 1) * every, pgd_steps)
        n_act += [int(active.sum().item())] * (nxt - t)
        if nxt >= pgd_steps:
            break
        P.pgd_run(X, nxt - t - 1, lr, mask=mask)
        Xp = X.clone()
        P.pgd_run(X, 1, lr, mask=mask)
        active &= (X != Xp).any(dim=1)
        t = nxt
    P.set_option(2, every)
    return np.asarray(n_act, dtype=np.int64)


def load_traffic(workload, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on `workload`, copied from an
    `ncu --set full` capture into profiles/traffic.csv (the capture and its command are named there); else None."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(path):
        return None
    try:
        import csv
        with open(path, newline="") as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload and row["kernel"] == kernel:
                    return int(row["dram_bytes_per_launch"])
    except Exception:
        return None
    return None


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm_gbs=float(p["hbm_gbs"]), sm_max_mhz=float(p.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


_FP32_PEAK = {}


def fp32_peak(device: int, peaks):
    """(measured, derived) plain-FP32 FMA peak in TFLOP/s.  Measured: the library's own FMA micro-benchmark kernel
    (afs_fp32_fma_peak: independent FFMA chains on every SM, best of 5, CUDA events) on this box, now; derived:
    148 SMs x 128 lanes x 2 flop x sm_max_mhz, the upper bound the measured figure is checked against."""
    if device not in _FP32_PEAK:
        import paper_2606_06656_b200 as afs
        _FP32_PEAK[device] = afs.fp32_fma_peak(device)
    return _FP32_PEAK[device], 148 * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12


# --------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        mhz, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            parts = [x.strip() for x in r.split(",")]
            if len(parts) < 6:
                continue
            try:
                mhz.append(float(parts[0])); mx = float(parts[1])
            except ValueError:
                continue
            for nm, val in zip(names, parts[2:6]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        return dict(sm_mhz=float(np.median(mhz)) if mhz else None, sm_max_mhz=mx, reasons=sorted(reasons),
                    samples=len(mhz))


# --------------------------------------------------------------------------------------------- oracle legs
def oracle_sample(inst, cfg, B_o=None, steps_o=None, target_s=8.0):
    """Time the oracle (as it stands) on a bounded sample: the first B_o restarts for steps_o PGD iterations.
    Unless given, the sample is sized from a one-iteration probe so that it costs about `target_s` seconds."""
    from oracle import ref
    cores = ref.num_threads()
    lr = float(np.float32(inst.lr))
    if B_o is None or steps_o is None:
        Bp = min(inst.B, cores)
        t0 = time.perf_counter()
        ref.pgd_run(inst, inst.X0[:Bp], 1, lr, mask=inst.mask)
        rate = Bp / max(time.perf_counter() - t0, 1e-6)            # restart-steps per second, rough
        B_o = min(inst.B, 32 * cores)
        steps_o = int(min(max(round(target_s * rate / B_o), 1), max(inst.steps, 1)))
        if steps_o == 1:
            B_o = int(min(max(round(target_s * rate), cores), B_o))
    t0 = time.perf_counter()
    ref.pgd_run(inst, inst.X0[:B_o], steps_o, lr, mask=inst.mask)
    dt = time.perf_counter() - t0
    return dict(value=B_o * steps_o / dt, seconds=dt, cores=cores, B_o=B_o, steps_o=steps_o)


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg = HEADLINE if args.config is None else args.config     # the workload the CUDA arm's headline names
    inst = W.config(cfg)
    from oracle import ref
    for _ in range(args.warmup):
        oracle_sample(inst, cfg, B_o=min(inst.B, 8), steps_o=1)
    tot_units, tot_t, last = 0.0, 0.0, None
    for _ in range(args.steps):
        last = oracle_sample(inst, cfg)
        tot_units += last["B_o"] * last["steps_o"]
        tot_t += last["seconds"]
    value = tot_units / tot_t
    sample = "configs[%d] instance, first %d restarts x %d PGD iterations per bench step" % (cfg, last["B_o"], last["steps_o"])
    line = dict(metric="pgd_restart_steps_per_sec", value=value, unit="restart-steps/s", n_gpus=args.gpus,
                steps=args.steps, warmup=args.warmup, ms_per_step=1e3 * tot_t / args.steps, higher_is_better=True,
                scaling="weak", vs_baseline=None, dtype="f64", data="synthetic", impl="reference",
                config=dict(workload=inst.name, n=inst.n, m=inst.m, nnz=inst.nnz, B=last["B_o"],
                            pgd_steps_per_call=last["steps_o"]),
                literal_evals_per_sec=value * inst.nnz,
                cpu_baseline=dict(value=value, unit="restart-steps/s", cores=ref.num_threads(), kind="oracle", sample=sample),
                e2e=dict(value=value, unit="restart-steps/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line))
    return 0


# --------------------------------------------------------------------------------------------- CUDA arm
def measure_config(cfg, args, afs, shard, rank, world, local, peaks):
    """Time configs[cfg]: `value` (device-resident inputs, CUDA events), `e2e` (host buffers through afs_pgd_run_host),
    the roofline of its dominant kernel and of the whole PGD iteration, and the oracle beside it.  Returns the JSON
    line of that configuration (rank 0; other ranks return None after taking part in the collectives)."""
    import torch
    import torch.distributed as dist

    inst = W.config(cfg)
    if world > 1:   # every rank its own start points (weak scaling), same instance
        inst.X0 = shard.rank_start_points(W.BASE_SEED, cfg, rank, inst.X0.shape)
    pgd_steps = inst.steps if args.pgd_steps is None else args.pgd_steps
    lr = float(np.float32(inst.lr))
    P = afs.Problem.from_instance(inst, device=local)
    # bench.py restates the library's class rules to attribute work to kernels: fail loudly if the two ever drift apart
    cls_here = kernel_class_of_constraints(inst)
    counts_here = {"var": int((cls_here == "var").sum()), "med0": int((cls_here == "med0").sum()),
                   "cmed+long": int(((cls_here == "cmed") | (cls_here == "long")).sum())}
    counts_lib = {"var": P.info("n_pull"), "med0": P.info("n_med"), "cmed+long": P.info("n_long")}   # info 5 counts both EK / CARD classes
    if getattr(inst, "weights", None) is None:      # weighted short clauses leave the pull path
        assert counts_here == counts_lib, ("bench.py's class rules differ from the library's", counts_here, counts_lib)
    if args.mode is not None:
        P.set_option(0, args.mode)
    if args.retire_every is not None:
        P.set_option(2, args.retire_every)
    X0 = torch.from_numpy(inst.X0).cuda()
    X = torch.empty_like(X0)
    mask = None if inst.mask is None else torch.from_numpy(inst.mask).cuda()
    out = dict(best_assign=torch.empty((inst.B, inst.n), dtype=torch.int8, device="cuda"),
               best_sat=torch.empty(inst.B, dtype=torch.int32, device="cuda"),
               best_step=torch.empty(inst.B, dtype=torch.int32, device="cuda"))
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    stream = torch.cuda.current_stream()

    def one_call(timed):
        X.copy_(X0)
        flush.fill_(1)                      # L2 flush between calls, outside the timed events
        if timed:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
        P.pgd_run(X, pgd_steps, lr, mask=mask, out=out)
        if timed:
            e1.record(stream)
            return e0, e1
        return None

    for _ in range(max(args.warmup, 0)):
        one_call(False)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    torch.cuda.synchronize()
    wall0 = time.perf_counter()
    evs = [one_call(True) for _ in range(args.steps)]
    torch.cuda.synchronize()
    wall = time.perf_counter() - wall0
    if world > 1:
        dist.barrier()
    clocks = sampler.stop() if sampler else None
    dev_ms = sum(a.elapsed_time(b) for a, b in evs)
    launches = P.info("launches") * args.steps
    resident = P.info("resident")
    dev_ms = shard.max_over_ranks(dev_ms, device="cuda")
    # the one exchange of the sharded job: best counts of every rank
    _, job_best = shard.gather_best(out["best_sat"])
    units = float(inst.B) * pgd_steps * args.steps * world
    value = units / (dev_ms * 1e-3)

    # ---- e2e through the host entry point (pinned buffers; copies inside the timed region)
    Xh0 = torch.from_numpy(inst.X0).pin_memory()
    Xh = torch.empty_like(Xh0).pin_memory()
    hout = dict(best_assign=torch.empty((inst.B, inst.n), dtype=torch.int8).pin_memory(),
                best_sat=torch.empty(inst.B, dtype=torch.int32).pin_memory(),
                best_step=torch.empty(inst.B, dtype=torch.int32).pin_memory())
    mask_h = None if inst.mask is None else torch.from_numpy(inst.mask).pin_memory()
    e2e_t = 0.0
    n_e2e = max(1, min(args.steps, 3))
    for i in range(1 + n_e2e):
        Xh.copy_(Xh0)
        flush.fill_(1)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        P.pgd_run_host(Xh, pgd_steps, lr, mask=mask_h, out=hout)     # synchronises the stream before returning
        dt = time.perf_counter() - t0
        if i > 0:
            e2e_t += dt
    e2e_value = float(inst.B) * pgd_steps * n_e2e * world / shard.max_over_ranks(e2e_t, device="cuda")
    h2d = inst.B * inst.n * 4 + (inst.n if inst.mask is not None else 0)
    d2h = inst.B * inst.n * 4 + inst.B * inst.n + 8 * inst.B

    if rank != 0:
        P.close()
        return None

    # ---- roofline.  ONE rule for every class: the work of a PGD iteration is the work of the
    # restarts that are active in it.  `step.frac` divides that by the time of the timed call (retirement on);
    # `step.no_retire` is a second timed pass with retirement off (afs_set_option(2, 0)): full-batch work over
    # full-batch time; `step.static_formula` is SURVEY.md 8(d)'s state-independent count over the time of the timed call.
    RETIRE = 32 if args.retire_every is None else args.retire_every         # the period `value` ran with (library default 32)
    every = 0 if resident else RETIRE
    n_act = active_trace(P, X0, pgd_steps, lr, mask, every)
    act_mean = float(n_act.mean()) if len(n_act) else float(inst.B)
    work = algorithmic_work(inst, act_mean)                                 # active restarts only
    work_act_static = dict(work)                                            # ... before the counted flops replace 6 L K
    work_full = algorithmic_work(inst)                                      # every restart in every iteration
    fp32_meas, fp32_derived = fp32_peak(local, peaks)
    stride = max(1, pgd_steps // 64)

    def profile_pass(ncalls):
        """per-launch spans (CUDA events on the launching stream, every stride-th iteration) in a pass of its own, so
        that the events do not sit in `value`; returns ({class: [ms, launches]}, {class: counted flops})"""
        P.set_option(1, stride)
        prof, counted = {}, {}
        for _ in range(ncalls):
            one_call(False)
            for k, (ms, cnt) in P.profile_read().items():
                a = prof.setdefault(k, [0.0, 0]); a[0] += ms; a[1] += cnt
            for k, fl in P.profile_flops().items():      # state-dependent flops counted by the long-constraint kernels
                counted[k] = counted.get(k, 0.0) + fl
        P.set_option(1, 0)
        return prof, counted

    prof, counted = profile_pass(max(1, min(args.steps, 3)))
    # the launches that serve the LONG class in one iteration count as one kernel group
    grp = [k for k in prof if k.startswith("long") or k == "glong"]
    if grp:
        iters = max(prof[k][1] for k in grp)
        prof["long"] = [sum(prof[k][0] for k in grp), iters]
        long_parts = {k: round(prof[k][0] / prof[k][1] * 1e3, 2) for k in grp}      # mean us per launch
        for k in grp:
            del prof[k]
        if "var" in prof and "glong" in long_parts:      # the variable pass's span brackets k_glong too
            prof["var"][0] = max(prof["var"][0] - long_parts["glong"] * 1e-3 * prof["var"][1], 0.0)
        fl = sum(v for k, v in counted.items() if k.startswith("long"))
        counted = {"long": fl} if fl else {}
    else:
        long_parts = None
    # Long EK/CARD kernels: literals on the boundary of the cube (clipped iterates, fixed variables) are exact shifts
    # and cost no arithmetic, so their algorithmic flops are the 6 Leff Keff the kernels count at the iterates they
    # actually see (active restarts only, by construction); the state-independent 6 L K stays beside it as
    # `static_formula`.
    for k, fl in counted.items():
        if k in prof and prof[k][1] > 0 and k in work:
            work[k] = (fl / prof[k][1], work[k][1])
    if counted:
        step_f = work["step"][0] - sum(work_act_static[k][0] for k in counted if k in work_act_static) + \
            sum(work[k][0] for k in counted if k in work)
        work["step"] = (step_f, work["step"][1])
    # k_sat_pull runs on the library's second stream BESIDE the variable pass: its span overlaps the others and is
    # reported on its own, not added to the time of the iteration
    overlapped = {k: prof.pop(k) for k in ("sat_pull",) if k in prof}
    per_iter_s = dev_ms * 1e-3 / (args.steps * max(pgd_steps, 1))           # whole PGD iteration, this rank
    # Event records between the launches of one iteration keep them from running back to back, so the spans of the
    # profile pass add up to more than the iteration takes in the timed call.  Each group's launch duration is its span
    # scaled by (time of the iteration in the timed call) / (sum of the spans per sampled iteration) when that is < 1:
    # launch_ms x launches per call <= ms_per_step then holds by construction; the raw span stays beside it.
    sampled_iters = max((v[1] for k, v in prof.items() if k != "boundary"), default=0)
    span_sum_s = sum(v[0] for k, v in prof.items() if k != "boundary") * 1e-3 / max(sampled_iters, 1)
    scale = 1.0
    if not resident and span_sum_s > per_iter_s > 0:
        scale = per_iter_s / span_sum_s
    dom = max((k for k in prof if k != "boundary"), key=lambda k: prof[k][0], default=None)
    roof = dict(bound=None, achieved=None, peak=None, unit=None, frac=None, traffic=None)
    alu_src = ("afs_fp32_fma_peak: FFMA micro-benchmark measured on this GPU in this run (derived bound "
               "148 SMs x 128 lanes x 2 flop x %.0f MHz = %.2f)" % (peaks["sm_max_mhz"], fp32_derived))
    if dom is not None:
        raw_s = prof[dom][0] * 1e-3 / prof[dom][1]                          # mean event-timed span of one launch (group)
        if resident:                                                        # one launch: never longer than the call it is in
            scale = min(1.0, dev_ms * 1e-3 / args.steps / raw_s)
        dur_s = raw_s * scale
        if dom == "resident":                                               # one launch = every iteration of the call
            flops, hbm = work["step"][0] * pgd_steps, 2 * inst.B * inst.n * 4 + inst.nnz * 4
        else:
            flops, hbm = work.get(dom, (0.0, 0.0))
        t_alu, t_hbm = flops / (fp32_meas * 1e12), hbm / (peaks["hbm_gbs"] * 1e9)
        if t_alu >= t_hbm:
            roof.update(bound="alu", achieved=flops / dur_s / 1e12, peak=fp32_meas, unit="TFLOP/s", peak_source=alu_src,
                        peak_derived=fp32_derived)
        else:
            roof.update(bound="hbm", achieved=hbm / dur_s / 1e9, peak=peaks["hbm_gbs"], unit="GB/s",
                        peak_source="MEASURED_PEAKS.json hbm_gbs (%s)" % peaks["source"])
        roof["frac"] = roof["achieved"] / roof["peak"]
        roof["kernel"] = dom
        if dom == "long":
            roof["kernel_group_us_per_launch"] = long_parts
        roof["launch_ms"] = dur_s * 1e3
        roof["launch_ms_event_span"] = raw_s * 1e3
        roof["span_scale"] = scale
        roof["launches_timed"] = prof[dom][1]
        launches_per_call = 1 if dom == "resident" else pgd_steps
        assert roof["launch_ms"] * launches_per_call <= dev_ms / args.steps * 1.0001, "launch_ms x launches exceeds ms_per_step"
        roof["algorithmic_per_launch"] = dict(flops=flops, hbm_bytes=hbm, restarts="active (mean %.1f of %d)" % (act_mean, inst.B))
        if dom in counted and dom in work_full:
            sf0 = work_full[dom][0]
            roof["static_formula"] = dict(flops_per_launch=sf0, frac_alu=sf0 / dur_s / 1e12 / fp32_meas,
                                          note="6 L K on the unfixed literals of the whole batch, whatever the iterate; the kernel skips boundary literals and retired restarts")
        tot_ms = sum(v[0] for k, v in prof.items())
        roof["share_of_timed_launches"] = {k: round(v[0] / tot_ms, 4) for k, v in sorted(prof.items(), key=lambda kv: -kv[1][0])}
        if overlapped:
            roof["overlapped_side_stream_us_per_launch"] = {k: round(v[0] / max(v[1], 1) * 1e3, 2) for k, v in overlapped.items()}
        roof["traffic"] = load_traffic(inst.name, dom)
    # the whole PGD iteration against the same two ceilings (every kernel of the step, launch gaps included): the
    # figure BASELINE.json's ">= 50 % of its roofline" target is judged on
    def step_roof(sf, sb, t_iter):
        t_alu, t_hbm = sf / (fp32_meas * 1e12), sb / (peaks["hbm_gbs"] * 1e9)
        return dict(bound="alu" if t_alu >= t_hbm else "hbm", roofline_us=max(t_alu, t_hbm) * 1e6,
                    measured_us=t_iter * 1e6, frac=max(t_alu, t_hbm) / t_iter,
                    algorithmic_per_iteration=dict(flops=sf, hbm_bytes=sb))
    roof["step"] = step_roof(work["step"][0], work["step"][1], per_iter_s)
    roof["step"]["active_restarts"] = dict(mean=act_mean, of=int(inst.B), retire_every=every,
                                           at_iteration={str(t): int(n_act[t]) for t in sorted({0, pgd_steps // 10, pgd_steps // 4, pgd_steps // 2, pgd_steps - 1}) if 0 <= t < len(n_act)})
    s0 = work_full["step"][0]
    roof["step"]["static_formula"] = dict(flops=s0, hbm_bytes=work_full["step"][1],
                                          frac=max(s0 / (fp32_meas * 1e12), work_full["step"][1] / (peaks["hbm_gbs"] * 1e9)) / per_iter_s,
                                          note="SURVEY.md 8(d): every restart in every iteration, 6 L K for EK / CARD, over the time of the timed call")
    if not resident and pgd_steps >= 20:
        # where the time of the call goes: the same call cut short at a few lengths (the PGD map is deterministic, so
        # the first k iterations of every call are the same work); differences of the call times = cost of the
        # iterations in between, entry / exit layout changes included in the first range
        cuts = sorted({max(pgd_steps // 50, 1), pgd_steps // 5, pgd_steps // 2, pgd_steps})
        t_cut = []
        for k in cuts:
            ts = []
            for _ in range(2):
                X.copy_(X0); flush.fill_(1)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream); P.pgd_run(X, k, lr, mask=mask, out=out); e1.record(stream)
                torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            t_cut.append(min(ts))
        lo, phases = 0, {}
        for k, t_ms, t_prev in zip(cuts, t_cut, [0.0] + t_cut[:-1]):
            phases["%d-%d" % (lo, k)] = dict(us_per_iteration=round((t_ms - t_prev) * 1e3 / (k - lo), 2),
                                             mean_active_restarts=round(float(n_act[lo:k].mean()), 1))
            lo = k
        roof["step"]["phases"] = phases
    if not resident:
        # retirement off: the same call on the full batch for every iteration, timed the same way (CUDA events around
        # the call, L2 flushed before it); work = the full batch, the LONG class by its counted flops of THIS pass
        P.set_option(2, 0)
        one_call(False)
        torch.cuda.synchronize()
        nr = [one_call(True) for _ in range(max(1, min(args.steps, 2)))]
        torch.cuda.synchronize()
        nr_iter_s = sum(a.elapsed_time(b) for a, b in nr) * 1e-3 / (len(nr) * max(pgd_steps, 1))
        prof_nr, counted_nr = profile_pass(1)
        fl_nr = sum(v for k, v in counted_nr.items() if k.startswith("long"))
        it_nr = max((prof_nr[k][1] for k in prof_nr if k.startswith("long") or k == "glong"), default=0)
        sf_nr = work_full["step"][0]
        if fl_nr and it_nr and "long" in work_full:
            sf_nr = sf_nr - work_full["long"][0] + fl_nr / it_nr
        P.set_option(2, RETIRE)
        roof["step"]["no_retire"] = step_roof(sf_nr, work_full["step"][1], nr_iter_s)
    else:
        roof["step"]["no_retire"] = dict(note="the tile-resident kernel never retires: same figure as step.frac",
                                         frac=roof["step"]["frac"], measured_us=per_iter_s * 1e6)

    # ---- the oracle beside it (bounded sample, rank 0, N = 1 only)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        o = oracle_sample(inst, cfg)
        cpu = dict(value=o["value"], unit="restart-steps/s", cores=o["cores"], kind="oracle",
                   sample="first %d restarts x %d PGD iterations of configs[%d] (%.1f s)" % (o["B_o"], o["steps_o"], cfg, o["seconds"]))
    P.close()
    return dict(metric="pgd_restart_steps_per_sec", value=value, unit="restart-steps/s", n_gpus=world,
                steps=args.steps, warmup=args.warmup, ms_per_step=dev_ms / args.steps, higher_is_better=True,
                scaling="weak", vs_baseline=None, dtype="f32", data="synthetic",
                config=dict(workload=inst.name, n=inst.n, m=inst.m, nnz=inst.nnz, B=inst.B, pgd_steps_per_call=pgd_steps,
                            lr=inst.lr, masked_vars=int((inst.mask != 0).sum()) if inst.mask is not None else 0,
                            l2="flushed between calls (256 MiB write), outside the timed events",
                            path="resident" if resident else "streaming", parallelism="restarts x%d" % world),
                literal_evals_per_sec=value * inst.nnz,
                wall_ms_per_step=1e3 * wall / args.steps,
                gpu_launches=int(launches), best_sat_max=int(job_best[2]),
                e2e=dict(value=e2e_value, unit="restart-steps/s", h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h)),
                roofline=roof, cpu_baseline=cpu, clocks=clocks)


HEADLINE = 4                      # the largest single-GPU configuration (by work): configs[4]
ALL_CONFIGS = (1, 2, 3, 4)        # the configurations BASELINE.json's target is set on


def run_cuda(args):
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2606_06656_b200 import build as afs_build
    if rank == 0:
        afs_build.build()
    if world > 1:
        dist.barrier()
    import paper_2606_06656_b200 as afs
    from paper_2606_06656_b200 import shard

    peaks = load_peaks()
    cfgs = ALL_CONFIGS if args.config is None else (args.config,)
    lines = {}
    for cfg in cfgs:
        lines[cfg] = measure_config(cfg, args, afs, shard, rank, world, local, peaks)
        torch.cuda.empty_cache()
    if rank == 0:
        head = HEADLINE if HEADLINE in lines else cfgs[-1]
        line = dict(lines[head])
        if len(cfgs) > 1:
            keep = ("value", "unit", "ms_per_step", "literal_evals_per_sec", "gpu_launches", "e2e", "roofline",
                    "cpu_baseline", "clocks", "config")
            line["per_config"] = [dict(cfg=c, **{k: lines[c][k] for k in keep}) for c in cfgs]
            line["gpu_launches"] = int(sum(lines[c]["gpu_launches"] for c in cfgs))
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def spawn_ranks(args):
    """`python bench.py --gpus N` with N > 1 outside torchrun: start N ranks (one per GPU) through
    torch.distributed.run on this node and pass the output through; NCCL's communicator log stays on."""
    port = 29500 + os.getpid() % 2000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")
    return subprocess.call(cmd, env=env)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=None,
                    help="BASELINE.json configs index; default: configs[1-4] in one run, configs[4] as the headline")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--pgd-steps", type=int, default=None, help="override the configuration's PGD iteration count")
    ap.add_argument("--mode", type=int, default=None, help="afs_set_option(0, mode): 1 streaming, 2 resident")
    ap.add_argument("--retire-every", type=int, default=None,
                    help="afs_set_option(2, K): retire restarts at a fixed point every K iterations (0 never; default: the library's 32)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.gpus > 1 and "RANK" not in os.environ:
        return spawn_ranks(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
