#!/usr/bin/env python
"""bench.py -- owner-local Muon step (MatrixFSDP, arxiv/paper_2607_05895) on B200: latency, algorithmic Newton-Schulz
TFLOP/s, roofline fractions, with the fp64 oracle timed beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c5] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

One "step" = one pass of the whole hot path over one resident set: mfsdp_muon_step on every
owned matrix + mfsdp_adamw_tail_step on every owned tail.  Default workload: BASELINE.json config 5 (Llama-3-70B
shapes, 64-rank NS-flops plan, heaviest rank) -- the set the north_star's targets are quoted on; it fits one GPU.
With N > 1 ranks, GPU r runs the r-th heaviest rank's resident set of the same plan (independent units, no
collective: "the optimizer step contains no matrix all-gather, broadcast, or redistribute").

`value` = algorithmic NS flops of all ranks / max-over-ranks device time (TFLOP/s, symmetric-aware count
F_alg = K [m(m+1)n + m^2(m+1) + 2 m^2 n]); `ms_per_step` is the step latency, the other half of BASELINE's metric.
Prints ONE JSON line on rank 0.  At N = 1 the line also carries `other_configs`: BASELINE.json configs 1-4 and the
paper's own setting on config 5, measured after the headline's timed region in the same process.

`--gpus N` with N > 1 and no WORLD_SIZE in the environment: this process spawns the N ranks itself (one per GPU, the
same environment torch.distributed.run would set) and forwards rank 0's line; under torch.distributed.run it is one
of the ranks.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "owner_muon_step_ns_algorithmic_tflops"
UNIT = "TFLOP/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="c5", choices=["c1", "c2", "c3", "c4", "c5", "paper16l"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--paper-setting", action="store_true",
                    help="the paper's own Muon hyper-parameters (PAPER.md:121): momentum 0.5, 2 NS steps, lr 1e-3")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true")
    ap.add_argument("--shampoo", default=None, choices=["c1", "c2", "c3", "c4", "paper16l"],
                    help="time only the owner-local Shampoo step (PAPER.md:182) on this config and print its record "
                         "(the `other_configs` entry; used for profiling)")
    return ap.parse_args()


# ---- work counts ---------------------------------------------------------------------------
def ns_flops(rows, cols, K):
    """(F_alg, F_dense, F_tile): symmetric-aware, dense, and what the 128 x N tiling executes."""
    m, n = min(rows, cols), max(rows, cols)
    f_alg = K * (m * (m + 1) * n + m * m * (m + 1) + 2 * m * m * n)
    f_dense = K * (4 * m * m * n + 2 * m * m * m)
    return f_alg, f_dense


def elementwise_bytes(rows, cols, wbytes):
    n = rows * cols
    return dict(mom=n * (wbytes + 4 + 4 + 2), upd=n * (wbytes + 2 + wbytes))


def apply_setting(wl, args):
    """--paper-setting: "Muon uses lr 1e-3, weight decay 1e-2, momentum 0.5, 2 NS steps, match_rms_adamw"
    (second timed workload on the same descriptors); AdamW betas (0.9, 0.999)."""
    if args.paper_setting:
        wl.muon.update(momentum=0.5, ns_steps=2, lr=1e-3, weight_decay=1e-2)
        wl.adamw.update(beta2=0.999)
        wl.name += "+paper_setting(mu0.5,K2)"
    return wl


def ncu_traffic(workload):
    """(bytes, commit) of one Newton-Schulz launch: dram__bytes_read.sum + dram__bytes_write.sum of an `ncu --set full`
    capture of this same command, kept in profiles/ncu_traffic.csv as `workload,kernel,bytes,commit` -- `commit` is the
    git commit the capture was taken at (stated again in the profiles README of that round), printed beside the number
    so that a stale capture is visible.  (None, None) if absent."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(path):
        return None, None
    for line in open(path):
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 3 and f[0] == workload and f[1] == "k_ns_tc":
            try:
                return float(f[2]), (f[3] if len(f) > 3 else None)
            except ValueError:
                return None, None
    return None, None


def min_hbm_bytes(rows, cols, K):
    """minimal HBM bytes of the Newton-Schulz chain of one matrix, K (3 m n + 4 m^2) * 2."""
    m, n = min(rows, cols), max(rows, cols)
    return K * (3 * m * n + 4 * m * m) * 2


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], tc_burst=d["bf16_tflops"], tc_sustained=d.get("bf16_tflops_sustained",
                    d["bf16_tflops"]), src="measured (MEASURED_PEAKS.json)")
    return dict(hbm=6650.0, tc_burst=1590.0, tc_sustained=1400.0, src="fallback (B200_PROFILING.md)")


# ---- clocks during the timed region ----------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        sm.sort()
        return dict(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(mx), power_w_max=max(pw), samples=len(sm),
                    reasons=sorted(reasons))


# ---- the oracle on the host cores (cpu_baseline leg and --impl reference) ----------------------------------------------
def plan_for(wl, rank_override=None):
    """Resident set via the oracle planner (used by the reference arm, which must not touch the CUDA library)."""
    from oracle import planner as oplan
    r = wl.rank if rank_override is None else rank_override
    return oplan.plan(wl.params, wl.world, wl.policy, wl.metric, r)


ORACLE_BUDGET_FLOPS = 2.6e13      # dense fp64 flops of the cpu_baseline sample: on the headline set that is every distinct
                                  # shape, 1024 x 8192 and 8192 x 8192 for all five iterations and the dominant 28672 x 8192
                                  # (79 % of the step's flops) for one whole iteration; about 40 s of dgemm on 16 host cores
REFERENCE_TOTAL_FLOPS = 8.0e13    # --impl reference: budget of the whole run (all steps and the warm-up): a few minutes


def oracle_sample(wl, desc, budget_flops=ORACLE_BUDGET_FLOPS):
    """Per-shape sample for the fp64 oracle: ONE resident matrix per distinct shape, cheapest shape
    first, each run for as many whole Newton-Schulz iterations k <= K as the remaining budget affords (at least the
    cheapest shape in full).  A shape whose single iteration does not fit is reported as not sampled.  The figure is a
    RATE (flops executed / seconds), so no extrapolation is involved.  Returns [(desc, k)], [skipped shapes]."""
    import workloads
    K = wl.muon["ns_steps"]
    first = {}
    for d in desc:
        if d["role"] == workloads.ROLE_MATRIX:
            first.setdefault((d["rows"], d["cols"]), d)
    sample, skipped, left = [], [], float(budget_flops)
    for (r, c), d in sorted(first.items(), key=lambda kv: ns_flops(kv[0][0], kv[0][1], 1)[1]):
        per_iter = ns_flops(r, c, 1)[1]
        k = int(min(K, left // per_iter)) if sample else K
        if k >= 1:
            sample.append((d, k))
            left -= k * per_iter
        else:
            skipped.append((r, c))
    return sample, skipped


def time_oracle(wl, sample, steps=1):
    """Runs oracle.muon.muon_step as it stands on each sampled matrix (with its iteration count); returns
    (seconds per pass, algorithmic flops executed, cores)."""
    import numpy as np
    import torch
    import workloads
    from oracle import muon as omuon
    K = wl.muon["ns_steps"]
    hp = wl.muon
    tdt = workloads.TORCH_DTYPE[wl.dtype]
    inputs = []
    for d, k in sample:
        W = torch.from_numpy(workloads.weight(wl, d["param_id"], d["rows"], d["cols"])).to(tdt).to(torch.float64).numpy()
        G = torch.from_numpy(workloads.gradient(wl, d["param_id"], d["rows"], d["cols"], 0)).to(tdt).to(
            torch.float64).numpy()
        inputs.append((W, G, np.zeros_like(W), k))
    f_alg = sum(ns_flops(d["rows"], d["cols"], k)[0] for d, k in sample)
    times = []
    for _ in range(steps):
        t0 = time.perf_counter()
        for W, G, M, k in inputs:
            omuon.muon_step(W, G, M, lr=hp["lr"], weight_decay=hp["weight_decay"], momentum=hp["momentum"],
                            nesterov=bool(hp["nesterov"]), ns_steps=k, coeffs=(hp["a"], hp["b"], hp["c"]),
                            eps=hp["eps"], scale_mode=hp["scale_mode"])
        times.append(time.perf_counter() - t0)
    try:
        cores = len(os.sched_getaffinity(0))
    except AttributeError:
        cores = os.cpu_count()
    cores = min(cores, torch.get_num_threads()) if torch.get_num_threads() > 0 else cores
    return times, f_alg, cores


def sample_text(wl, sample, skipped, budget=None):
    budget = ORACLE_BUDGET_FLOPS if budget is None else budget
    K = wl.muon["ns_steps"]
    txt = "per-shape sampled, one matrix per distinct resident shape: " + ", ".join(
        "%dx%d (%d of %d NS iterations)" % (d["rows"], d["cols"], k, K) for d, k in sample)
    if skipped:
        txt += "; not affordable within %.1e fp64 flops: " % budget + ", ".join("%dx%d" % s for s in skipped)
    return txt


def workload_config(wl, descs, plan_rank):
    """The `config` object of the JSON line -- the same on both arms (the planners agree bit for bit)."""
    import workloads
    K = wl.muon["ns_steps"]
    mats = [d for d in descs if d["role"] == workloads.ROLE_MATRIX]
    tails = [d for d in descs if d["role"] == workloads.ROLE_TAIL]
    n_el = workloads.flat_elems(descs)[0]
    wbytes = 2 if wl.dtype == workloads.BF16 else 4
    return dict(workload=wl.name, plan_rank=plan_rank, matrices=len(mats), tails=len(tails), matrix_elems=int(n_el),
                ns_steps=K, l2="inputs larger than L2" if n_el * wbytes > 256e6 else
                "working set may fit L2 (not flushed)",
                ns_flops_alg=sum(ns_flops(d["rows"], d["cols"], K)[0] for d in mats),
                ns_flops_dense=sum(ns_flops(d["rows"], d["cols"], K)[1] for d in mats))


def run_reference(args):
    """--impl reference: the fp64 oracle, as it stands, on the host cores; each step the same bounded per-shape sample
    the cpu_baseline leg of our arm uses."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import workloads
    wl = apply_setting(workloads.get(args.config), args)
    pl = plan_for(wl)
    n_warm = max(0, min(args.warmup, 1))
    budget = min(ORACLE_BUDGET_FLOPS, REFERENCE_TOTAL_FLOPS / (max(1, args.steps) + n_warm))
    sample, skipped = oracle_sample(wl, pl["desc"], budget)
    for _ in range(n_warm):
        time_oracle(wl, sample, 1)
    times, f_alg, cores = time_oracle(wl, sample, max(1, args.steps))
    t = sum(times) / len(times)
    val = f_alg / t / 1e12
    txt = sample_text(wl, sample, skipped, budget)
    line = dict(impl="reference", metric=METRIC, value=val, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=t * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic (seeded, workloads/)", config=workload_config(wl, pl["desc"], pl["rank"]),
                cpu_baseline=dict(value=val, unit=UNIT, cores=cores, kind="oracle", sample=txt),
                e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


# ---- our arm -------------------------------------------------------------------------------------------------------------
def rank_order_by_load(mf, wl):
    """Ranks of the plan sorted by primary load, heaviest first (ties -> lowest id)."""
    pr = mf.mfsdp_plan(wl.params, wl.world, wl.policy, wl.metric, 0)
    loads = pr.rank_load[:wl.world]
    return sorted(range(wl.world), key=lambda r: (-loads[r], r))


def choose_plan_rank(order, wl_rank, rank, world):
    """Which rank of the plan this process runs: at N = 1 the workload's own choice (heaviest when wl_rank < 0); at
    N > 1 process r takes the r-th heaviest rank (independent resident sets, no collective on the data path)."""
    if world > 1 or wl_rank < 0:
        return order[rank % len(order)]
    return wl_rank


def reduce_over_ranks(ms, ms_e2e, f_alg, launches, world, device):
    """MAX over ranks of the device times, SUM over ranks of flops and launches (the only collective: the report)."""
    import torch
    import torch.distributed as dist
    stats = torch.tensor([ms, ms_e2e, float(f_alg), float(launches)], dtype=torch.float64, device=device)
    if world > 1:
        mx = stats.clone(); dist.all_reduce(mx, op=dist.ReduceOp.MAX)
        sm = stats.clone(); dist.all_reduce(sm, op=dist.ReduceOp.SUM)
        return mx[0].item(), mx[1].item(), sm[2].item(), int(sm[3].item())
    return ms, ms_e2e, float(f_alg), int(launches)


def ev_time(torch, stream, fn, reps):
    """Mean device time (ms) of fn() over reps, CUDA events recorded on `stream`, synchronised on both sides."""
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(reps):
        fn()
    e1.record(stream)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


class Resident:
    """One resident set on the current device: plan, seeded inputs in pinned host memory and in HBM, workspace."""

    def __init__(self, mf, wl, plan_rank, pin=True):
        import torch
        import workloads
        self.mf, self.wl, self.plan_rank = mf, wl, plan_rank
        pr = mf.mfsdp_plan(wl.params, wl.world, wl.policy, wl.metric, plan_rank)
        self.desc = pr.desc
        self.descs = [self.desc[i] for i in range(self.desc._n)]
        self.ddicts = [d.as_dict() for d in self.descs]
        self.mats = [d for d in self.descs if d.role == mf.ROLE_MATRIX]
        self.tails = [d for d in self.descs if d.role == mf.ROLE_TAIL]
        self.K = wl.muon["ns_steps"]
        self.hp = mf.MuonHParams(precision=wl.precision, **wl.muon)
        self.n_mat_el, self.n_tail_el = mf.mfsdp_flat_elems(self.desc)
        self.wbytes = 2 if wl.dtype == mf.BF16 else 4
        self.hW = workloads.fill_flat(wl, self.descs, workloads.KIND_W, pin=pin)
        self.hG = workloads.fill_flat(wl, self.descs, workloads.KIND_G, step=0, pin=pin)
        self.W, self.G = self.hW.cuda(), self.hG.cuda()
        self.M = torch.zeros(self.n_mat_el, dtype=torch.float32, device="cuda")
        self.P = workloads.fill_flat(wl, self.descs, workloads.KIND_W, role=mf.ROLE_TAIL).cuda()
        self.Gt = workloads.fill_flat(wl, self.descs, workloads.KIND_G, role=mf.ROLE_TAIL).cuda()
        self.m1 = torch.zeros(self.n_tail_el, dtype=torch.float32, device="cuda")
        self.v1 = torch.zeros(self.n_tail_el, dtype=torch.float32, device="cuda")
        ws_bytes = mf.mfsdp_workspace_bytes(self.desc, wl.precision)
        raw = torch.empty(ws_bytes + 1024, dtype=torch.uint8, device="cuda")
        off = (-raw.data_ptr()) % 1024
        self.ws = raw[off:off + ws_bytes]
        self._raw = raw
        self.stream = torch.cuda.current_stream()
        self.t = 0
        self.f_alg = sum(ns_flops(d.rows, d.cols, self.K)[0] for d in self.mats)
        self.f_dense = sum(ns_flops(d.rows, d.cols, self.K)[1] for d in self.mats)

    def set_hparams(self, muon, adamw):
        import copy
        self.wl = copy.deepcopy(self.wl)              # the caller's workload object keeps its own setting
        self.wl.muon.update(muon)
        self.wl.adamw.update(adamw)
        self.K = self.wl.muon["ns_steps"]
        self.hp = self.mf.MuonHParams(precision=self.wl.precision, **self.wl.muon)
        self.f_alg = sum(ns_flops(d.rows, d.cols, self.K)[0] for d in self.mats)
        self.f_dense = sum(ns_flops(d.rows, d.cols, self.K)[1] for d in self.mats)

    def step(self):
        """One pass of the whole hot path: mfsdp_muon_step on every owned matrix + mfsdp_adamw_tail_step on the tails."""
        mf = self.mf
        self.t += 1
        mf.mfsdp_muon_step(self.desc, self.W, self.G, self.M, self.ws, self.hp, self.stream)
        if self.tails:
            mf.mfsdp_adamw_tail_step(self.desc, self.P, self.Gt, self.m1, self.v1,
                                     mf.AdamWHParams(step=self.t, **self.wl.adamw), self.stream)

    def time_steps(self, torch, steps, barrier):
        n0 = self.mf.mfsdp_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(self.stream)
        for _ in range(steps):
            self.step()
        e1.record(self.stream)
        barrier()
        return e0.elapsed_time(e1) / steps, self.mf.mfsdp_launch_count() - n0

    def time_passes(self, torch, reps):
        """Device time of each pass on its own (CUDA events on the launching stream).  The Newton-Schulz pass is the
        dominant kernel; inside mfsdp_muon_step its last epilogue also applies the weight update when that is fused."""
        mf, st = self.mf, self.stream
        t = dict(mom=ev_time(torch, st, lambda: mf.mfsdp_muon_momentum_pass(self.desc, self.G, self.M, self.ws, self.hp, st), reps),
                 ns=ev_time(torch, st, lambda: mf.mfsdp_muon_ns_pass(self.desc, self.ws, self.hp, st), reps),
                 upd=ev_time(torch, st, lambda: mf.mfsdp_muon_update_pass(self.desc, self.W, self.ws, self.hp, st), reps),
                 adam=ev_time(torch, st, lambda: mf.mfsdp_adamw_tail_step(
                     self.desc, self.P, self.Gt, self.m1, self.v1, mf.AdamWHParams(step=self.t + 1, **self.wl.adamw), st),
                     reps) if self.tails else 0.0)
        return t

    def byte_counts(self):
        b_mom = sum(elementwise_bytes(d.rows, d.cols, self.wbytes)["mom"] for d in self.mats)
        b_upd = sum(elementwise_bytes(d.rows, d.cols, self.wbytes)["upd"] for d in self.mats)
        b_adam = sum(d.rows * d.cols for d in self.tails) * (3 * self.wbytes + 16)
        return b_mom, b_upd, b_adam


def passes_record(res, t, pk):
    b_mom, b_upd, b_adam = res.byte_counts()
    gbs = lambda b, ms: b / (ms * 1e-3) / 1e9 if ms else 0.0
    return dict(momentum=dict(ms=t["mom"], gbs=gbs(b_mom, t["mom"]), frac_hbm=gbs(b_mom, t["mom"]) / pk["hbm"]),
                update=dict(ms=t["upd"], gbs=gbs(b_upd, t["upd"]), frac_hbm=gbs(b_upd, t["upd"]) / pk["hbm"],
                            note="separate pass; mfsdp_muon_step applies the update in the last NS epilogue when "
                                 "the weights are bf16 and every cols % 8 == 0"),
                adamw=dict(ms=t["adam"], gbs=gbs(b_adam, t["adam"])), ns=dict(ms=t["ns"]))


def compact_config(rec, pk):
    """One row of roofline.configs from a verbose other_configs record: the numbers the documents quote, nothing else."""
    if "error" in rec:
        return dict(workload=rec.get("workload"), error=rec["error"][:120])
    if "refresh_step" in rec:           # Shampoo: the method's own work is fp32-class; three-term operands issue 6 x that in bf16
        peak = pk["tc_sustained"] if rec["frac_of"].startswith("sustained") else pk["tc_burst"]
        f32 = rec["refresh_step"]["f32_class_tflops"]
        return dict(workload=rec["workload"] + "+shampoo", bound="tensor", unit="TFLOP/s (fp32-class)", achieved=f32,
                    peak=peak / 6.0, frac=f32 / (peak / 6.0), frac_of=rec["frac_of"].split(" ")[0] + " bf16 peak / 6",
                    issued_bf16_tflops=rec["refresh_step"]["umma_bf16_tflops"], refresh_ms=rec["refresh_step"]["ms"],
                    stale_ms=rec["stale_step"]["ms"], root_iters_max=rec["refresh_step"]["root_iters_max"],
                    sm_mhz=rec["clocks"]["sm_mhz"])
    return dict(workload=rec["workload"], ms_per_step=rec["ms_per_step"], ns_ms=rec["ns_ms"], ns_tflops_alg=rec["ns_tflops_alg"],
                ns_frac=rec["ns_frac"], frac_of=rec["ns_frac_of"].split(" ")[0], momentum_gbs=rec["momentum_gbs"],
                update_gbs=rec["update_gbs"], launches_per_step=rec["launches_per_step"], sm_mhz=rec["clocks"]["sm_mhz"])


def measure_other_config(torch, mf, name, pk, local, paper=False, reuse=None, precision=None):
    """One record of `other_configs`: the same step on another BASELINE.json config (or the paper's own setting on the
    headline's resident set), timed long enough to be meaningful (>= 0.3 s or 200 steps), clocks sampled alongside."""
    import workloads
    if reuse is None:
        wl = workloads.get(name)
        if precision is not None:      # e.g. config 1 (fp32 storage) through the bf16 tensor-core Newton-Schulz kernels
            wl.precision = precision
            wl.name += "+ns_bf16" if precision == mf.NS_BF16 else "+ns_fp32"
        res = Resident(mf, wl, choose_plan_rank(rank_order_by_load(mf, wl), wl.rank, 0, 1), pin=False)
    else:
        res = reuse
    if paper:
        res.set_hparams(dict(momentum=0.5, ns_steps=2, lr=1e-3, weight_decay=1e-2), dict(beta2=0.999))
    for _ in range(3):
        res.step()
    torch.cuda.synchronize()
    ms0, _ = res.time_steps(torch, 3, torch.cuda.synchronize)
    steps = int(max(5, min(200, 0.3e3 / max(ms0, 1e-3))))
    sampler = ClockSampler(local)
    sampler.start()
    ms, launches = res.time_steps(torch, steps, torch.cuda.synchronize)
    t = res.time_passes(torch, max(3, min(steps, 50)))
    clocks = sampler.stop()
    capped = "sw_power_cap" in clocks.get("reasons", [])
    peak = pk["tc_sustained"] if capped else pk["tc_burst"]
    ns_tf = res.f_alg / (t["ns"] * 1e-3) / 1e12
    rec = dict(workload=res.wl.name + ("+paper_setting(mu0.5,K2)" if paper else ""), ms_per_step=ms, steps=steps,
               ns_ms=t["ns"], ns_tflops_alg=ns_tf, ns_frac=ns_tf / peak,
               ns_frac_of="sustained bf16 peak (sw_power_cap sampled)" if capped else "burst bf16 peak",
               precision="bf16" if res.wl.precision == mf.NS_BF16 else "f32 (FFMA correctness mode)",
               momentum_gbs=passes_record(res, t, pk)["momentum"]["gbs"], update_gbs=passes_record(res, t, pk)["update"]["gbs"],
               launches_per_step=launches / steps, clocks=dict(sm_mhz=clocks.get("sm_mhz"), reasons=clocks.get("reasons")),
               l2="inputs larger than L2" if res.n_mat_el * res.wbytes > 256e6 else
               "working set may fit L2 (not flushed): steady-state optimizer-step latency of a set this small")
    return rec


def measure_shampoo(torch, mf, name, pk, local, ws_cap_bytes=64e9):
    """One record of `other_configs` for the owner-local Shampoo step on a
    BASELINE.json config: step 1 recomputes every inverse fourth root (root_every = 2), step 2 reuses them.  Flops are
    counted from the iteration counts the device reports: fp32-class flops (symmetric products count once) and the
    bf16 UMMA flops actually issued for them (x6 for three-term operands, x3 / x2 for the two-term preconditioning
    products, x1 for the statistics of a bf16 gradient),
    the latter against the bf16 tensor peak."""
    import numpy as np
    import workloads
    wl = workloads.get(name)
    pr = mf.mfsdp_plan(wl.params, wl.world, wl.policy, wl.metric, choose_plan_rank(rank_order_by_load(mf, wl), wl.rank, 0, 1))
    desc = pr.desc
    descs = [desc[i] for i in range(desc._n)]
    mats = [d for d in descs if d.role == mf.ROLE_MATRIX]

    def aligned(nbytes):
        raw = torch.empty(nbytes + 1024, dtype=torch.uint8, device="cuda")
        off = (-raw.data_ptr()) % 1024
        out = raw[off:off + nbytes]
        out._keep = raw
        return out
    state = aligned(mf.mfsdp_shampoo_state_bytes(desc))
    state.zero_()
    lo, hi = mf.mfsdp_shampoo_workspace_bytes(desc, 0)
    ws = aligned(int(max(lo, min(hi, ws_cap_bytes))))
    W = workloads.fill_flat(wl, descs, workloads.KIND_W).cuda()
    gt = 1 if wl.dtype == mf.BF16 else 3
    stream = torch.cuda.current_stream()
    sampler = ClockSampler(local)
    sampler.start()
    recs = []
    G = None
    for t in (1, 2):
        hG = workloads.fill_flat(wl, descs, workloads.KIND_G, step=t)
        if G is None:
            G = hG.cuda()
        else:
            G.copy_(hG)      # same gradient buffer every step, as in training: the launch tables are keyed by its address
        torch.cuda.synchronize()
        n0 = mf.mfsdp_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        mf.mfsdp_shampoo_step(desc, W, G, state, ws, mf.ShampooHParams(step=t, root_every=2), stream)
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        f32 = umma = 0.0
        iters = []
        for i, d in enumerate(mats):
            v = mf.mfsdp_shampoo_view(desc, 0, i)
            raw = ws[v[9]: v[9] + 2 * v[10]].cpu().numpy().tobytes()
            for k, dd in enumerate((d.rows, d.cols)):
                it = int(np.frombuffer(raw[k * v[10] + 36: k * v[10] + 40], dtype=np.uint32)[0])
                iters.append(it)
                if t == 1:
                    f32 += it * 4.0 * dd ** 3                    # four symmetric d x d x d products per iteration
                    umma += it * 4.0 * dd ** 3 * 6
            stat = float(d.rows) * d.rows * d.cols + float(d.cols) * d.cols * d.rows
            p1, p2 = 2.0 * d.rows * d.rows * d.cols, 2.0 * d.rows * d.cols * d.cols
            f32 += stat + p1 + p2
            umma += stat * gt * (gt + 1) / 2 + p1 * (2 if gt == 1 else 3) + p2 * 3      # S4 runs on two-term operands
        recs.append(dict(ms=ms, launches=mf.mfsdp_launch_count() - n0, f32_class_tflops=f32 / ms / 1e9,
                         umma_bf16_tflops=umma / ms / 1e9, root_iters_max=max(iters), root_iters_mean=float(np.mean(iters))))
    clocks = sampler.stop()
    capped = "sw_power_cap" in clocks.get("reasons", [])
    peak = pk["tc_sustained"] if capped else pk["tc_burst"]
    return dict(workload=wl.name, optimizer="owner-local Shampoo (PAPER.md:182): full L / R, inverse fourth roots by coupled "
                "Newton, fp32-class GEMMs as three-term bf16 on tcgen05", refresh_step=recs[0], stale_step=recs[1],
                refresh_frac_of_bf16_peak=recs[0]["umma_bf16_tflops"] / peak,
                frac_of="sustained bf16 peak (sw_power_cap sampled)" if capped else "burst bf16 peak",
                state_gb=state.numel() / 1e9, workspace_gb=ws.numel() / 1e9, n_matrices=len(mats),
                clocks=dict(sm_mhz=clocks.get("sm_mhz"), reasons=clocks.get("reasons")))


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2607_05895_b200 as mf
    import workloads

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (sm_100a); there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    mf.load()

    if args.shampoo:
        print(json.dumps(measure_shampoo(torch, mf, args.shampoo, peaks(), local)))
        return
    wl = apply_setting(workloads.get(args.config), args)
    order = rank_order_by_load(mf, wl)
    plan_rank = choose_plan_rank(order, wl.rank, rank, world)
    res = Resident(mf, wl, plan_rank)
    stream = res.stream

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        res.step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    ms, launches = res.time_steps(torch, args.steps, barrier)
    # per-pass device times inside the same clock-sampled window (dominant kernel: the Newton-Schulz pass)
    t = res.time_passes(torch, max(3, min(args.steps, 10)))
    clocks = sampler.stop()

    # e2e: the same step through the HOST-buffer C-ABI entry point (pinned host W, G, M up; W, M back), every step
    ms_e2e = 0.0
    if not args.no_e2e:
        hM = torch.zeros(max(res.n_mat_el, 1), dtype=torch.float32, pin_memory=True)[:res.n_mat_el]
        dW, dG, dM = torch.empty_like(res.W), torch.empty_like(res.G), torch.empty_like(res.M)
        n_e2e = max(2, min(args.steps, 3))
        hws_bytes = mf.mfsdp_host_workspace_bytes(res.desc, wl.precision)      # one workspace slice per pipelined group
        if hws_bytes > res.ws.numel():
            raw = torch.empty(hws_bytes + 1024, dtype=torch.uint8, device="cuda")
            off = (-raw.data_ptr()) % 1024
            res.ws, res._raw = raw[off:off + hws_bytes], raw
        mf.mfsdp_muon_step_host(res.desc, res.hW, res.hG, hM, dW, dG, dM, 1, res.ws, res.hp, stream)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record(stream)
        for _ in range(n_e2e):
            mf.mfsdp_muon_step_host(res.desc, res.hW, res.hG, hM, dW, dG, dM, 1, res.ws, res.hp, stream)
        e1.record(stream)
        barrier()
        ms_e2e = max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3) / n_e2e
        # the same call with the optimizer state resident in HBM (upload_state = 0): only the step's input G goes up,
        # W and M still come back every step.  Reported beside the headline e2e, which moves the state both ways.
        ms_e2e_res = ms_e2e_mom = 0.0
        if world == 1:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0 = time.perf_counter()
            e0.record(stream)
            for _ in range(n_e2e):
                mf.mfsdp_muon_step_host(res.desc, res.hW, res.hG, hM, dW, dG, dM, 0, res.ws, res.hp, stream)
            e1.record(stream)
            barrier()
            ms_e2e_res = max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3) / n_e2e
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0 = time.perf_counter()
            e0.record(stream)
            for _ in range(n_e2e):       # upload_state = 2: the momentum never leaves the device (G up, W down)
                mf.mfsdp_muon_step_host(res.desc, res.hW, res.hG, hM, dW, dG, dM, 2, res.ws, res.hp, stream)
            e1.record(stream)
            barrier()
            ms_e2e_mom = max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3) / n_e2e
        del dW, dG, dM, hM

    ms_all, ms_e2e_all, f_all, launches_all = reduce_over_ranks(ms, ms_e2e, res.f_alg, launches, world, "cuda")
    per_rank = [ms]
    if world > 1:
        every = [torch.zeros(2, dtype=torch.float64, device="cuda") for _ in range(world)]
        dist.all_gather(every, torch.tensor([ms, float(plan_rank)], dtype=torch.float64, device="cuda"))
        per_rank = [float(x[0].item()) for x in every]
        ranks_run = [int(x[1].item()) for x in every]
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    pk = peaks()
    value = f_all / (ms_all * 1e-3) / 1e12
    ns_tflops = res.f_alg / (t["ns"] * 1e-3) / 1e12
    cfg = workload_config(wl, res.ddicts, plan_rank)
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
                ms_per_step=ms_all, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="bf16" if
                wl.precision == mf.NS_BF16 else "f32", data="synthetic (seeded, workloads/)", config=cfg,
                gpu_launches=launches_all, clocks=clocks)
    traffic, traffic_commit = ncu_traffic(wl.name)
    min_bytes = sum(min_hbm_bytes(d.rows, d.cols, res.K) for d in res.mats)
    line["roofline"] = dict(bound="tensor", kernel="k_ns_tc (one launch per tile class walks all iterations and phases)",
                            achieved=ns_tflops, peak=pk["tc_sustained"], unit="TFLOP/s",
                            frac=ns_tflops / pk["tc_sustained"], traffic=traffic, traffic_commit=traffic_commit,
                            traffic_ratio=(traffic / min_bytes) if traffic else None, min_hbm_bytes=min_bytes,
                            peak_source=pk["src"] + ", sustained bf16", frac_of_burst=ns_tflops / pk["tc_burst"],
                            dense_equiv_tflops=res.f_dense / (t["ns"] * 1e-3) / 1e12, ms=t["ns"])
    line["roofline"]["passes"] = passes_record(res, t, pk)      # the HBM-bound passes of the same step, against the copy peak
    if world > 1:
        pr = mf.mfsdp_plan(wl.params, wl.world, wl.policy, wl.metric, 0)
        planned = [pr.rank_load[r] for r in ranks_run]
        line["per_rank"] = dict(plan_ranks=ranks_run, ms=per_rank,
                                imbalance_measured=max(per_rank) * len(per_rank) / sum(per_rank),
                                imbalance_planned=max(planned) * len(planned) / max(1, sum(planned)))
    if not args.no_e2e:
        h2d = res.n_mat_el * (2 * res.wbytes + 4)
        d2h = res.n_mat_el * (res.wbytes + 4)
        line["e2e"] = dict(value=f_all / (ms_e2e_all * 1e-3) / 1e12, unit=UNIT, ms_per_step=ms_e2e_all,
                           h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h),
                           api="mfsdp_muon_step_host (pinned host W, G, M; resident set pipelined in groups)")
        if world == 1 and ms_e2e_res > 0.0:
            line["e2e"]["state_resident"] = dict(ms_per_step=ms_e2e_res, value=f_all / (ms_e2e_res * 1e-3) / 1e12,
                                                 h2d_bytes_per_step=int(res.n_mat_el * res.wbytes),
                                                 d2h_bytes_per_step=int(d2h),
                                                 note="upload_state = 0: W and M stay in HBM between steps, G up, W and M down")
            line["e2e"]["momentum_on_device"] = dict(ms_per_step=ms_e2e_mom, value=f_all / (ms_e2e_mom * 1e-3) / 1e12,
                                                     h2d_bytes_per_step=int(res.n_mat_el * res.wbytes),
                                                     d2h_bytes_per_step=int(res.n_mat_el * res.wbytes),
                                                     note="upload_state = 2: optimizer state resident in HBM, G up, W down")
    if world == 1 and not args.no_other_configs and args.config == "c5" and not args.paper_setting:
        others = []
        try:
            others.append(measure_other_config(torch, mf, "c5", pk, local, paper=True, reuse=res))
        except Exception as e:      # a failed side measurement must not lose the headline
            others.append(dict(workload="c5+paper_setting", error=repr(e)))
        del res
        torch.cuda.empty_cache()
        for name in ("c1", "c2", "c3", "c4", "paper16l"):
            try:      # paper16l: the paper's own Table 1 / 3 workload (one rank's share) with the paper's own setting
                others.append(measure_other_config(torch, mf, name, pk, local, paper=(name == "paper16l")))
            except Exception as e:
                others.append(dict(workload=name, error=repr(e)))
            torch.cuda.empty_cache()
        try:      # config 1 is defined in fp32 mode (an FFMA correctness mode here); the same set on the tensor-core path
            others.append(measure_other_config(torch, mf, "c1", pk, local, precision=mf.NS_BF16))
        except Exception as e:
            others.append(dict(workload="c1+ns_bf16", error=repr(e)))
        for name in ("c2", "c4"):
            try:
                others.append(measure_shampoo(torch, mf, name, pk, local))
            except Exception as e:
                others.append(dict(workload=name + "+shampoo", error=repr(e)))
            torch.cuda.empty_cache()
        line["other_configs"] = others
        line["roofline"]["configs"] = [compact_config(o, pk) for o in others]
    if not args.no_cpu_baseline and world == 1:
        desc_d = plan_for(wl, plan_rank)["desc"]
        sample, skipped = oracle_sample(wl, desc_d)
        times, fa, cores = time_oracle(wl, sample, 1)
        line["cpu_baseline"] = dict(value=fa / times[0] / 1e12, unit=UNIT, cores=cores, kind="oracle",
                                    sample=sample_text(wl, sample, skipped), seconds=times[0])
    # key order: the verbose per-config records first, the compact blocks (roofline with its `configs` and `passes`,
    # cpu_baseline, e2e) last, so that a consumer that keeps only the tail of the line still holds every quoted number
    for key in ("e2e", "cpu_baseline", "roofline"):
        if key in line:
            line[key] = line.pop(key)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def spawn_ranks(args):
    """`python bench.py --gpus N` without torch.distributed.run: start the N ranks here (one process per GPU, NCCL
    only for the report), forward rank 0's JSON line.  The path has no data-path collective."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    procs = []
    for r in range(args.gpus):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(args.gpus), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, os.path.abspath(__file__)] + sys.argv[1:], env=env,
                                      stdout=subprocess.PIPE if r == 0 else subprocess.DEVNULL, text=True))
    out, _ = procs[0].communicate()
    rc = procs[0].returncode
    for p_ in procs[1:]:
        rc = rc or p_.wait()
    sys.stdout.write(out)
    sys.stdout.flush()
    if rc:
        raise SystemExit(rc)


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
