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
Prints ONE JSON line on rank 0.
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
    ap.add_argument("--config", default="c5", choices=["c1", "c2", "c3", "c4", "c5"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--paper-setting", action="store_true",
                    help="the paper's own Muon hyper-parameters (PAPER.md:121): momentum 0.5, 2 NS steps, lr 1e-3")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
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
    """DRAM bytes of one k_ns_tc launch (dram__bytes_read.sum + dram__bytes_write.sum of an `ncu --set full` capture of
    this same command), copied by hand into profiles/ncu_traffic.csv: lines `workload,kernel,bytes`.  None if absent."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(path):
        return None
    for line in open(path):
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 3 and f[0] == workload and f[1] == "k_ns_tc":
            try:
                return float(f[2])
            except ValueError:
                return None
    return None


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


def oracle_sample(wl, desc, budget_flops=2.5e12):
    """A bounded sample of the resident set for the fp64 oracle: resident matrices, cheapest NS cost first, until
    ~budget_flops dense fp64 flops (about 10-30 s of dgemm on the host cores); at least one matrix."""
    import workloads
    K = wl.muon["ns_steps"]
    mats = [d for d in desc if d["role"] == workloads.ROLE_MATRIX]
    sample, acc = [], 0.0
    for d in sorted(mats, key=lambda d: ns_flops(d["rows"], d["cols"], K)[1]):
        f = ns_flops(d["rows"], d["cols"], K)[1]
        if sample and acc + f > budget_flops:
            break
        sample.append(d); acc += f
    return sample


def time_oracle(wl, sample, steps=1):
    """Runs oracle.muon.muon_step as it stands on each sampled matrix; returns (seconds per pass, F_alg, cores)."""
    import numpy as np
    import torch
    import workloads
    from oracle import muon as omuon
    K = wl.muon["ns_steps"]
    hp = wl.muon
    tdt = workloads.TORCH_DTYPE[wl.dtype]
    inputs = []
    for d in sample:
        W = torch.from_numpy(workloads.weight(wl, d["param_id"], d["rows"], d["cols"])).to(tdt).to(torch.float64).numpy()
        G = torch.from_numpy(workloads.gradient(wl, d["param_id"], d["rows"], d["cols"], 0)).to(tdt).to(
            torch.float64).numpy()
        inputs.append((W, G, np.zeros_like(W)))
    f_alg = sum(ns_flops(d["rows"], d["cols"], K)[0] for d in sample)
    times = []
    for _ in range(steps):
        t0 = time.perf_counter()
        for W, G, M in inputs:
            omuon.muon_step(W, G, M, lr=hp["lr"], weight_decay=hp["weight_decay"], momentum=hp["momentum"],
                            nesterov=bool(hp["nesterov"]), ns_steps=K, coeffs=(hp["a"], hp["b"], hp["c"]),
                            eps=hp["eps"], scale_mode=hp["scale_mode"])
        times.append(time.perf_counter() - t0)
    try:
        cores = len(os.sched_getaffinity(0))
    except AttributeError:
        cores = os.cpu_count()
    cores = min(cores, torch.get_num_threads()) if torch.get_num_threads() > 0 else cores
    return times, f_alg, cores


def sample_text(sample):
    shapes = {}
    for d in sample:
        shapes[(d["rows"], d["cols"])] = shapes.get((d["rows"], d["cols"]), 0) + 1
    return "cheapest resident matrices: " + ", ".join("%d x %dx%d" % (n, r, c) for (r, c), n in shapes.items())


def run_reference(args):
    """--impl reference: the fp64 oracle, as it stands, on the host cores; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import workloads
    wl = apply_setting(workloads.get(args.config), args)
    pl = plan_for(wl)
    sample = oracle_sample(wl, pl["desc"], budget_flops=1.0e12)
    for _ in range(max(0, min(args.warmup, 1))):
        time_oracle(wl, sample, 1)
    times, f_alg, cores = time_oracle(wl, sample, max(1, args.steps))
    t = sum(times) / len(times)
    val = f_alg / t / 1e12
    line = dict(impl="reference", metric=METRIC, value=val, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=t * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic (seeded, workloads/)",
                config=dict(workload=wl.name, sample=sample_text(sample), ns_steps=wl.muon["ns_steps"]),
                cpu_baseline=dict(value=val, unit=UNIT, cores=cores, kind="oracle", sample=sample_text(sample)),
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

    wl = apply_setting(workloads.get(args.config), args)
    order = rank_order_by_load(mf, wl)
    plan_rank = choose_plan_rank(order, wl.rank, rank, world)
    pr = mf.mfsdp_plan(wl.params, wl.world, wl.policy, wl.metric, plan_rank)
    desc = pr.desc
    descs = [desc[i] for i in range(desc._n)]
    mats = [d for d in descs if d.role == mf.ROLE_MATRIX]
    tails = [d for d in descs if d.role == mf.ROLE_TAIL]
    K = wl.muon["ns_steps"]
    hp = mf.MuonHParams(precision=wl.precision, **wl.muon)
    n_mat_el, n_tail_el = mf.mfsdp_flat_elems(desc)
    tdt = workloads.TORCH_DTYPE[wl.dtype]
    wbytes = 2 if wl.dtype == mf.BF16 else 4

    # seeded inputs, generated on the host, resident in pinned memory (e2e leg) and copied to HBM (device leg)
    hW = workloads.fill_flat(wl, descs, workloads.KIND_W, pin=True)
    hG = workloads.fill_flat(wl, descs, workloads.KIND_G, step=0, pin=True)
    hM = torch.zeros(max(n_mat_el, 1), dtype=torch.float32, pin_memory=True)[:n_mat_el]
    W, G, M = hW.cuda(), hG.cuda(), torch.zeros(n_mat_el, dtype=torch.float32, device="cuda")
    P = workloads.fill_flat(wl, descs, workloads.KIND_W, role=mf.ROLE_TAIL).cuda()
    Gt = workloads.fill_flat(wl, descs, workloads.KIND_G, role=mf.ROLE_TAIL).cuda()
    m1 = torch.zeros(n_tail_el, dtype=torch.float32, device="cuda")
    v1 = torch.zeros(n_tail_el, dtype=torch.float32, device="cuda")
    ws_bytes = mf.mfsdp_workspace_bytes(desc, wl.precision)
    raw = torch.empty(ws_bytes + 1024, dtype=torch.uint8, device="cuda")
    off = (-raw.data_ptr()) % 1024
    ws = raw[off:off + ws_bytes]
    stream = torch.cuda.current_stream()
    tstep = [0]

    def step():
        tstep[0] += 1
        mf.mfsdp_muon_step(desc, W, G, M, ws, hp, stream)
        if tails:
            mf.mfsdp_adamw_tail_step(desc, P, Gt, m1, v1, mf.AdamWHParams(step=tstep[0], **wl.adamw), stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    n0 = mf.mfsdp_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    launches = mf.mfsdp_launch_count() - n0
    ms = e0.elapsed_time(e1) / args.steps

    # per-pass device times inside the same clock-sampled window (dominant kernel: the Newton-Schulz pass)
    reps = max(3, min(args.steps, 10))
    t_mom = ev_time(torch, stream, lambda: mf.mfsdp_muon_momentum_pass(desc, G, M, ws, hp, stream), reps)
    t_ns = ev_time(torch, stream, lambda: mf.mfsdp_muon_ns_pass(desc, ws, hp, stream), reps)
    t_upd = ev_time(torch, stream, lambda: mf.mfsdp_muon_update_pass(desc, W, ws, hp, stream), reps)
    t_adam = ev_time(torch, stream, lambda: mf.mfsdp_adamw_tail_step(
        desc, P, Gt, m1, v1, mf.AdamWHParams(step=tstep[0] + 1, **wl.adamw), stream), reps) if tails else 0.0
    clocks = sampler.stop()

    # e2e: the same step through the HOST-buffer C-ABI entry point (pinned host W, G, M up; W, M back), every step
    ms_e2e = 0.0
    if not args.no_e2e:
        dW, dG, dM = torch.empty_like(W), torch.empty_like(G), torch.empty_like(M)
        hM.zero_()
        n_e2e = max(2, min(args.steps, 3))
        mf.mfsdp_muon_step_host(desc, hW, hG, hM, dW, dG, dM, 1, ws, hp, stream)
        barrier()
        t0 = time.perf_counter()
        e0.record(stream)
        for _ in range(n_e2e):
            mf.mfsdp_muon_step_host(desc, hW, hG, hM, dW, dG, dM, 1, ws, hp, stream)
        e1.record(stream)
        barrier()
        ms_e2e = max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3) / n_e2e
        del dW, dG, dM
    f_alg = sum(ns_flops(d.rows, d.cols, K)[0] for d in mats)
    f_dense = sum(ns_flops(d.rows, d.cols, K)[1] for d in mats)
    b_mom = sum(elementwise_bytes(d.rows, d.cols, wbytes)["mom"] for d in mats)
    b_upd = sum(elementwise_bytes(d.rows, d.cols, wbytes)["upd"] for d in mats)
    b_adam = sum(d.rows * d.cols for d in tails) * (3 * wbytes + 16)

    ms_all, ms_e2e_all, f_all, launches_all = reduce_over_ranks(ms, ms_e2e, f_alg, launches, world, "cuda")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    pk = peaks()
    value = f_all / (ms_all * 1e-3) / 1e12
    ns_tflops = f_alg / (t_ns * 1e-3) / 1e12
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
                ms_per_step=ms_all, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="bf16" if
                wl.precision == mf.NS_BF16 else "f32", data="synthetic (seeded, workloads/)",
                config=dict(workload=wl.name, plan_rank=plan_rank, matrices=len(mats), tails=len(tails),
                            matrix_elems=int(n_mat_el), ns_steps=K, l2="inputs larger than L2" if
                            n_mat_el * wbytes > 256e6 else "working set may fit L2 (not flushed)",
                            ns_flops_alg=f_alg, ns_flops_dense=f_dense),
                gpu_launches=launches_all, clocks=clocks)
    line["roofline"] = dict(bound="tensor", kernel="k_ns_tc (one launch per tile class walks all iterations and phases)",
                            achieved=ns_tflops, peak=pk["tc_sustained"], unit="TFLOP/s",
                            frac=ns_tflops / pk["tc_sustained"], traffic=ncu_traffic(wl.name),
                            peak_source=pk["src"] + ", sustained bf16", frac_of_burst=ns_tflops / pk["tc_burst"],
                            dense_equiv_tflops=f_dense / (t_ns * 1e-3) / 1e12, ms=t_ns)
    line["passes"] = dict(
        momentum=dict(ms=t_mom, gbs=b_mom / (t_mom * 1e-3) / 1e9, frac_hbm=b_mom / (t_mom * 1e-3) / 1e9 / pk["hbm"]),
        update=dict(ms=t_upd, gbs=b_upd / (t_upd * 1e-3) / 1e9, frac_hbm=b_upd / (t_upd * 1e-3) / 1e9 / pk["hbm"]),
        adamw=dict(ms=t_adam, gbs=(b_adam / (t_adam * 1e-3) / 1e9) if t_adam else 0.0), ns=dict(ms=t_ns))
    if not args.no_e2e:
        h2d = n_mat_el * (2 * wbytes + 4)
        d2h = n_mat_el * (wbytes + 4)
        line["e2e"] = dict(value=f_all / (ms_e2e_all * 1e-3) / 1e12, unit=UNIT, ms_per_step=ms_e2e_all,
                           h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h),
                           api="mfsdp_muon_step_host (pinned host W, G, M)")
    if not args.no_cpu_baseline and world == 1:
        sample = oracle_sample(wl, [d.as_dict() | dict(role=d.role) for d in descs])
        times, fa, cores = time_oracle(wl, sample, 1)
        line["cpu_baseline"] = dict(value=fa / times[0] / 1e12, unit=UNIT, cores=cores, kind="oracle",
                                    sample=sample_text(sample), seconds=times[0])
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
