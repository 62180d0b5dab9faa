#!/usr/bin/env python
"""bench.py -- headline benchmark of libtnrd on B200:  Mpixel-stages/s of the 48-filter 7x7, T=5 TNRD model.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--size 4096] [--T 5]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 ... bench.py --gpus N

A "step" is one pass of the whole hot path (rows a1-a6 of DESIGN.md: one tnrd_diffuse call = 2 staging launches + T
stage launches of the tensor-core kernel) over one synthetic noisy image of BASELINE.json configs[3] (size x size, sigma 25).  One process
per GPU; with N > 1 every rank runs the same workload on its own image (independent problems, no data-path
collective -> weak scaling); the time is the max over ranks of a CUDA-event interval bracketed by barrier +
synchronize.  Prints ONE JSON line on rank 0.

--impl reference times the CPU oracle (oracle/, as it stands) on the box's host cores on a bounded sample of
the same workload; see DESIGN.md "Measurement".
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
sys.path.insert(0, ROOT)

import tnrd_gen  # noqa: E402

METRIC = "Mpixel-stages/s"
N_K, KSIZE, M = 48, 7, 63                          # headline model; main() re-derives them per workload
EX2_PER_PX_STAGE = N_K * M                       # 3024 MUFU.EX2 per pixel-stage (direct phi)
FMA_PER_PX_STAGE = 2 * N_K * KSIZE * KSIZE       # 4704 FFMA of filtering
FLOP_PER_PX_STAGE = 2 * FMA_PER_PX_STAGE + 5 * EX2_PER_PX_STAGE   # per RBF term: sub, mul, ex2, fma(2) -> 24528
NOMINAL_SM_MHZ, NOMINAL_SMS, MUFU_PER_CLK_SM, FMA_PER_CLK_SM = 1965.0, 148, 16, 128
# factorised phi, tile kernel: 5 groups of 13 centres; per response and group 3 ex2 and
# 16 FMA-pipe operations (add, 2 mul, 12 Horner FMAs, 1 FMA into the sum)
FACT_GROUPS, FACT_EX2_PER_GROUP, FACT_FMA_PER_GROUP = 5, 3, 16
# factorised phi, tensor-core kernel: per response 2 ex2 (rho0, 1/rho0) + 2 FMA-pipe
# operations, per group 1 ex2 and 17 FMA-pipe operations (add, d^2, two rho scalings, 12 Horner FMAs, 1 into the sum);
# + 2 per response for the BF16 hi/lo split of v.  The filterings run on the tensor pipe: forward 3 TF32 passes of
# K = 8 ks (window of 8 columns per tap row) x N = 2 N_k per pixel pair, scatter 2 BF16 passes of K = 4 N_k x N = 8 (ks + 1)
TC_EX2_PER_RESP, TC_EX2_PER_GROUP, TC_FMA_PER_RESP, TC_FMA_PER_GROUP = 2, 1, 4, 17
TF32_MAC_PER_CLK_SM, BF16_MAC_PER_CLK_SM = 1024 * 2, 1024 * 4        # nominal dense: 1.1 / 2.25 PFLOP/s over 148 SMs at 1.9 GHz
# dram__bytes_* per launch of the dominant kernel come from the ncu launch list committed under profiles/ (written by
# the ncu command named in profiles/r02_launches.md for THIS library version); absent or stale -> null
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r02_dram_stage.csv")


def read_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


class ClockSampler:
    """Samples nvidia-smi SM clock and throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *exc):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
                for nm, val in zip(names, r[3:7]):
                    if val.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        # keep samples taken under load (clock above idle); fall back to all samples
        busy = [c for c in sm if c > 0.6 * mx] or sm
        return {"sm_mhz": float(np.median(busy)) if busy else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


def measured_traffic(kernel_substr: str, lib_version: int):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the kernels whose name contains kernel_substr, from the
    CSV the committed ncu command wrote (profiles/r02_dram_stage.csv; the command and the library version it profiled are
    in profiles/r02_launches.md).  None unless both files exist and the .md names this library version."""
    try:
        import csv
        md = open(os.path.join(ROOT, "profiles", "r02_launches.md")).read()
        if f"tnrd_version={lib_version}" not in md:
            return None
        lines = [ln for ln in open(TRAFFIC_CSV).read().splitlines() if ln.startswith('"')]
        per = {}
        for r in csv.DictReader(lines):
            if kernel_substr in r.get("Kernel Name", "") and r.get("Metric Name", "").startswith("dram__bytes_"):
                v = float(r["Metric Value"].replace(",", ""))
                v *= {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(r.get("Metric Unit", "byte"), 1.0)
                per[r["ID"]] = per.get(r["ID"], 0.0) + v
        return float(np.mean(list(per.values()))) if per else None
    except Exception:
        return None


def oracle_sample(cfg, cores_hint=None, target_s=12.0):
    """Time the oracle on a bounded crop of the workload; returns (Mpx-stages/s, cores, sample text, seconds)."""
    import oracle
    cores = oracle.num_threads()
    T = cfg["T"]
    per_core = 20e-6                                   # measured on the B200 host: ~20 us per 48x7x7 px-stage per core
    px = max(48 * 48, int(target_s * cores / per_core / T))
    side = int(min(cfg["H"], cfg["W"], max(48, int(px ** 0.5))))
    y0, x0 = (cfg["H"] - side) // 2, (cfg["W"] - side) // 2
    f = cfg["f"][0, y0:y0 + side, x0:x0 + side]
    t0 = time.perf_counter()
    out = oracle.diffuse(f, f, cfg["filters"], cfg["rbf_w"], cfg["rbf_mu"], cfg["rbf_gamma"], cfg["lambda"])
    dt = time.perf_counter() - t0
    assert np.all(np.isfinite(out))
    val = side * side * T / dt / 1e6
    return val, cores, f"centre {side}x{side} crop of the {cfg['H']}x{cfg['W']} image, all T={T} stages, {dt:.1f} s", dt


def run_reference(args, rank):
    """--impl reference: the oracle as it stands on the host cores; rank 0 only."""
    if rank != 0:
        return
    cfg = tnrd_gen.make_config(4, size=args.size, T=args.T)
    vals, secs, sample, cores = [], [], "", 1
    for i in range(args.warmup + args.steps):
        v, cores, sample, dt = oracle_sample(cfg, target_s=args.ref_seconds)
        if i >= args.warmup:
            vals.append(v); secs.append(dt)
    value = float(np.mean(vals))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "Mpixel-stages/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(secs)),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"C4 {args.size}x{args.size} T={args.T} N_k=48 7x7 (BASELINE.json configs[3])",
                   "sample": sample},
        "cpu_baseline": {"value": value, "unit": "Mpixel-stages/s", "cores": cores, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": "Mpixel-stages/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4", choices=["c1", "c2", "c3", "c4", "c5", "deblock", "backward"],
                    help="BASELINE.json config; c4 (default) is the headline, the others are for exploration")
    ap.add_argument("--size", type=int, default=4096)
    ap.add_argument("--T", type=int, default=5)
    ap.add_argument("--ref-seconds", type=float, default=10.0, help="CPU seconds per oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--kernel", default="auto", choices=["auto", "tile", "tc"],
                    help="stage kernel (tnrd_set_kernel): auto (default), the tile kernel, the tensor-core kernel; profiling")
    ap.add_argument("--no-window", action="store_true", help="skip the extra windowed-phi measurement")
    ap.add_argument("--shard", default="images", choices=["images", "slab"],
                    help="N > 1: 'images' = one image per GPU (weak scaling, default); 'slab' = ONE image split into row "
                         "slabs with a 2rT overlap, no exchange (strong scaling; c4 only)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    import paper_1503_05768_b200 as tnrd
    from paper_1503_05768_b200.shard import max_over_ranks, sum_over_ranks

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the TNRD hot path has no CPU fallback")
    tnrd.build()
    tnrd.lib()
    kernel_sel = {"auto": tnrd.KERNEL_AUTO, "tile": tnrd.KERNEL_TILE, "tc": tnrd.KERNEL_TC}[args.kernel]
    tnrd.tnrd_set_kernel(kernel_sel)
    torch.cuda.set_device(local_rank)
    devs = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=devs)
    warmup = max(args.warmup, 3)

    deblock = args.workload == "deblock"
    backward = args.workload == "backward"   # joint-training step: T forward stages + back-propagation, all gradients
    if backward:
        args.workload, args.no_window = "c4", True
        if args.size == 4096:
            args.size = 2048                 # keeps the P/V maps of the filter gradient at 1.6 GB
    if deblock:      # TRD^4_{7x7} JPEG deblocking at 1024^2, the size the paper times it at
        cfg = tnrd_gen.make_deblock(9, 1, 1024, 1024, 4, 48, 7)
        cfg["f"], cfg["lambda"] = cfg["u0"], np.zeros(4, dtype=np.float32)
        args.no_window = True
    else:
        cfg = (tnrd_gen.make_config(4, size=args.size, T=args.T) if args.workload == "c4"
               else tnrd_gen.make_config(int(args.workload[1])))
    own_rows = cfg["H"]
    slab = args.shard == "slab" and world > 1 and args.workload == "c4" and not deblock and not backward
    if slab:    # this rank's rows of the one image, with the 2 r T margin it needs (paper_1503_05768_b200/shard.py)
        from paper_1503_05768_b200.shard import slab_bounds
        lo, hi, s0, s1 = slab_bounds(cfg["H"], rank, world, cfg["T"], cfg["ksize"])
        cfg = dict(cfg, H=s1 - s0, f=np.ascontiguousarray(cfg["f"][:, s0:s1]), u0=np.ascontiguousarray(cfg["u0"][:, s0:s1]))
        own_rows = hi - lo
    B, H, W, T = cfg["B"], cfg["H"], cfg["W"], cfg["T"]
    N_K, KSIZE = cfg["N_k"], cfg["ksize"]
    EX2_PER_PX_STAGE, FMA_PER_PX_STAGE = N_K * M, 2 * N_K * KSIZE * KSIZE
    FLOP_PER_PX_STAGE = 2 * FMA_PER_PX_STAGE + 5 * EX2_PER_PX_STAGE
    f = torch.from_numpy(cfg["f"]).to(devs)
    out = torch.empty_like(f)
    k, w = torch.from_numpy(cfg["filters"]).to(devs), torch.from_numpy(cfg["rbf_w"]).to(devs)
    mu, lam = torch.from_numpy(cfg["rbf_mu"]).to(devs), torch.from_numpy(cfg["lambda"]).to(devs)
    gamma = cfg["rbf_gamma"]
    stream = torch.cuda.current_stream()

    if deblock:
        qlo, qhi = torch.from_numpy(cfg["qcs_lo"]).to(devs), torch.from_numpy(cfg["qcs_hi"]).to(devs)

    if backward:
        gt = torch.from_numpy(cfg["clean"]).to(devs) if "clean" in cfg else f * 0.98
        g_u0, g_k, g_w, g_l = torch.empty_like(f), torch.empty_like(k), torch.empty_like(w), torch.empty_like(lam)

    def step():
        if backward:
            tnrd.tnrd_diffuse_backward(f, f, gt, None, B, H, W, T, N_K, KSIZE, k, w, mu, gamma, lam, out, g_u0, g_k, g_w,
                                       g_l, stream)
        elif deblock:
            tnrd.tnrd_deblock_diffuse(f, B, H, W, T, N_K, KSIZE, k, w, mu, gamma, qlo, qhi, out, stream)
        else:
            tnrd.tnrd_diffuse(f, f, B, H, W, T, N_K, KSIZE, k, w, mu, gamma, lam, out, stream)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        step()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    tnrd.tnrd_reset_launch_count()
    with ClockSampler(local_rank) as clocks:      # the timed region: K steps between two events, nothing else on the stream
        e0.record(stream)
        for i in range(args.steps):
            step()
        e1.record(stream)
        barrier()
    launches = tnrd.tnrd_launch_count()
    ms = max_over_ranks(e0.elapsed_time(e1), devs)
    # per-step marks for the median and the best step, in a pass of their own: an event between two 15 us launches costs
    # as much as a third of a launch, so the marks stay out of the timed region
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    marks[0].record(stream)
    for i in range(args.steps):
        step()
        marks[i + 1].record(stream)
    barrier()
    step_ms = sorted(marks[i].elapsed_time(marks[i + 1]) for i in range(args.steps))
    ms_median, ms_best = float(np.median(step_ms)), float(step_ms[0])
    px_stages_all = sum_over_ranks(float(B) * own_rows * W * T * args.steps, devs)     # output pixels only
    value = px_stages_all / (ms * 1e-3) / 1e6

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region -------------
    hf = torch.from_numpy(cfg["f"]).pin_memory()
    hout = torch.empty_like(hf).pin_memory()
    hp = [cfg["filters"], cfg["rbf_w"], cfg["rbf_mu"], cfg["lambda"]]

    if deblock:
        hq = [torch.from_numpy(cfg["qcs_lo"]).pin_memory(), torch.from_numpy(cfg["qcs_hi"]).pin_memory()]
        dq = [torch.empty_like(f), torch.empty_like(f), torch.empty_like(f), torch.empty_like(f)]

    if backward:
        hgt = gt.cpu().pin_memory()
        hg = [torch.empty(g_k.shape).pin_memory(), torch.empty(g_w.shape).pin_memory(), torch.empty(g_l.shape).pin_memory()]
        dgt = torch.empty_like(f)

    def step_host():
        if backward:  # host f, u_gt up; parameter gradients and u_T down
            dq0 = out  # reuse
            f.copy_(hf, non_blocking=True); dgt.copy_(hgt, non_blocking=True)
            tnrd.tnrd_diffuse_backward(f, f, dgt, None, B, H, W, T, N_K, KSIZE, k, w, mu, gamma, lam, dq0, None, g_k, g_w,
                                       g_l, stream)
            hout.copy_(dq0, non_blocking=True)
            hg[0].copy_(g_k, non_blocking=True); hg[1].copy_(g_w, non_blocking=True); hg[2].copy_(g_l, non_blocking=True)
            stream.synchronize()
        elif deblock:   # no host entry point for this variant: explicit pinned copies around the device call
            dq[0].copy_(hf, non_blocking=True); dq[1].copy_(hq[0], non_blocking=True); dq[2].copy_(hq[1], non_blocking=True)
            tnrd.tnrd_deblock_diffuse(dq[0], B, H, W, T, N_K, KSIZE, k, w, mu, gamma, dq[1], dq[2], dq[3], stream)
            hout.copy_(dq[3], non_blocking=True)
            stream.synchronize()
        else:
            tnrd.tnrd_diffuse_host(hf, hf, B, H, W, T, N_K, KSIZE, hp[0], hp[1], hp[2], gamma, hp[3], hout, stream)

    step_host()
    barrier()
    e2e_steps = max(1, min(args.steps, 5))
    e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2.record(stream)
    for _ in range(e2e_steps):
        step_host()
    e3.record(stream)
    barrier()
    ms_e2e = max_over_ranks(e2.elapsed_time(e3), devs)
    e2e_value = sum_over_ranks(float(B) * own_rows * W * T * e2e_steps, devs) / (ms_e2e * 1e-3) / 1e6
    h2d = hf.numel() * 4 * (3 if deblock else 2 if backward else 1) + (0 if deblock or backward else sum(int(a.nbytes) for a in hp))
    d2h = hout.numel() * 4 + (sum(x.numel() * 4 for x in hg) if backward else 0)
    same = bool(torch.equal(hout.to(devs), out))

    # ---- extra: the other phi evaluators, same workload, same timing protocol: direct (tnrd_set_phi_mode(0)) ... ------
    win = None
    tile = None
    if not args.no_window:
        def timed():
            for _ in range(warmup):
                step()
            barrier()
            ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ea.record(stream)
            for _ in range(args.steps):
                step()
            eb.record(stream)
            barrier()
            return max_over_ranks(ea.elapsed_time(eb), devs)
        # the same (default, factorised) evaluator on the tile kernel: what the tensor-core kernel replaced
        tnrd.tnrd_set_kernel(tnrd.KERNEL_TILE)
        ms_t = timed()
        tile_out = out.clone()
        tnrd.tnrd_set_kernel(kernel_sel)
        tile = px_stages_all / (ms_t * 1e-3) / 1e6
        tnrd.tnrd_set_phi_mode(0)
        for _ in range(warmup):
            step()
        barrier()
        direct_out = out.clone()
        e8, e9 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e8.record(stream)
        for _ in range(args.steps):
            step()
        e9.record(stream)
        barrier()
        ms_d = max_over_ranks(e8.elapsed_time(e9), devs)
        direct = px_stages_all / (ms_d * 1e-3) / 1e6
        # ... windowed (tnrd_set_phi_mode(1)) ...
        tnrd.tnrd_set_phi_mode(1)
        for _ in range(warmup):
            step()
        barrier()
        e4, e5 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e4.record(stream)
        for _ in range(args.steps):
            step()
        e5.record(stream)
        barrier()
        ms_w = max_over_ranks(e4.elapsed_time(e5), devs)
        win = px_stages_all / (ms_w * 1e-3) / 1e6
        # ... and the lookup-table evaluator (tnrd_set_phi_mode(2): the authors' own approximation)
        tnrd.tnrd_set_phi_mode(2)
        for _ in range(warmup):
            step()
        barrier()
        lut_out = out.clone()
        e6, e7 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e6.record(stream)
        for _ in range(args.steps):
            step()
        e7.record(stream)
        barrier()
        tnrd.tnrd_set_phi_mode(tnrd.PHI_FACTORED)
        lut = px_stages_all / (max_over_ranks(e6.elapsed_time(e7), devs) * 1e-3) / 1e6
        step(); barrier()
        lut_dist = float((lut_out - out).abs().max())
        direct_dist = float((direct_out - out).abs().max())
        tile_dist = float((tile_out - out).abs().max())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel ---------------------------------------------------------------------------
    # Which stage kernel the library used for this shape (include/tnrd.h: tnrd_tc_plan_query): the tensor-core kernel
    # (stage_tc_kernel) or the tile kernel (stage_fused_kernel).  Both are plain-ALU bound: the declared counts of the
    # formulation each implements give one time per pipe, the largest is the roofline (SURVEY.md 8d accounting rule).
    sms = torch.cuda.get_device_properties(devs).multi_processor_count
    tcq = tnrd.tnrd_tc_plan_query(B, H, W, N_K, KSIZE, sms)
    use_tc = (tcq["applies"] == 2 and args.kernel == "auto") or (tcq["applies"] >= 1 and args.kernel == "tc")
    # one launch per tnrd_diffuse call = the small-image kernel (all stages in one launch; include/tnrd.h tnrd_set_kernel)
    use_small = (not deblock and not backward) and launches == args.steps
    if use_small:
        use_tc = False
    launch_s = (ms * 1e-3) / (args.steps * T)           # step time / T: the staging kernels (~us) are charged too
    fma_peak = NOMINAL_SMS * FMA_PER_CLK_SM * NOMINAL_SM_MHZ * 1e6 / 1e12
    xu_peak = NOMINAL_SMS * MUFU_PER_CLK_SM * NOMINAL_SM_MHZ * 1e6 / 1e12
    mb = {n: tnrd.tnrd_microbench(i) / 1e12 for i, n in enumerate(["ffma_T_per_s", "ex2_T_per_s", "phi_terms_T_per_s"])}
    px_per_launch = float(B) * H * W
    executed_frac = None
    if use_tc:
        # executed vs defined phi work: one extra, untimed step with the library's counters on
        tnrd.tnrd_phi_stats(True)
        step()
        ex, de = tnrd.tnrd_phi_stats(False)
        executed_frac = ex / de if de else None
        e = executed_frac if executed_frac is not None else 1.0
        fma_def = N_K * (TC_FMA_PER_RESP + FACT_GROUPS * TC_FMA_PER_GROUP)
        fma_exe = N_K * (TC_FMA_PER_RESP + e * FACT_GROUPS * TC_FMA_PER_GROUP)
        ex2_def = N_K * (TC_EX2_PER_RESP + FACT_GROUPS * TC_EX2_PER_GROUP)
        ex2_exe = N_K * (TC_EX2_PER_RESP + e * FACT_GROUPS * TC_EX2_PER_GROUP)
        nkp = (N_K + 7) // 8 * 8
        mac_tf32 = 3 * (8 * KSIZE) * (2 * nkp) / 2.0               # per pixel: 3 passes, K = 8 ks, N = 2 N_k, 2 pixels per row of M
        mac_bf16 = 2 * (4 * nkp) * (8 * (KSIZE + 1)) / 2.0
        clk = {"fma": fma_def / FMA_PER_CLK_SM, "xu": ex2_def / MUFU_PER_CLK_SM,
               "tensor": mac_tf32 / TF32_MAC_PER_CLK_SM + mac_bf16 / BF16_MAC_PER_CLK_SM}
        kernel_name, form = "stage_tc_kernel", "tensor-core kernel: filterings on tcgen05 (TF32 x3 forward, BF16 hi/lo scatter), factorised phi with one exponential pair per response"
        tensor_extra = {"tf32_mac_per_px_stage": mac_tf32, "bf16_mac_per_px_stage": mac_bf16,
                        "tensor_clk_per_px_sm_nominal": clk["tensor"]}
    else:
        fma_def = fma_exe = N_K * (2 * KSIZE * KSIZE + FACT_GROUPS * FACT_FMA_PER_GROUP)
        ex2_def = ex2_exe = N_K * FACT_GROUPS * FACT_EX2_PER_GROUP
        clk = {"fma": fma_def / FMA_PER_CLK_SM, "xu": ex2_def / MUFU_PER_CLK_SM, "tensor": 0.0}
        kernel_name, form = "stage_fused_kernel", "tile kernel: filterings and factorised phi on the FMA pipe (dead groups skipped, not counted)"
        tensor_extra = {}
    bound_pipe = max(clk, key=clk.get)                          # the pipe the declared counts load most
    roof_clk = clk[bound_pipe]                                   # clocks per pixel-stage per SM at 100 % of that pipe
    roof_value = NOMINAL_SMS * NOMINAL_SM_MHZ * 1e6 / roof_clk / 1e6      # Mpixel-stages/s if all DEFINED work ran at peak
    achieved = fma_exe * px_per_launch / launch_s / 1e12        # EXECUTED FMA-pipe operations per second
    backward_or_deblock = backward or deblock
    roofline = {
        "bound": "alu", "pipe": "fma (FFMA2/FMUL2/FADD2)" if bound_pipe == "fma" else bound_pipe, "kernel": kernel_name,
        "formulation": form,
        "achieved": None if backward else achieved, "peak": fma_peak, "unit": "Tfma/s",
        "frac": None if backward else achieved / fma_peak,
        "traffic": measured_traffic(kernel_name, tnrd.tnrd_version()) if (args.workload == "c4" and H == W == 4096 and T == 5
                                                                         and not backward_or_deblock) else None,
        "traffic_source": "profiles/r02_dram_stage.csv (ncu launch list of this command, see profiles/r02_launches.md)",
        "peak_source": "148 SM x 128 FMA-pipe lanes/clk/SM x 1.965 GHz (DESIGN.md Roofline; no FP32 peak in MEASURED_PEAKS.json); "
                       f"measured by tnrd_microbench: {mb['ffma_T_per_s']:.3f} Tfma/s",
        "fma_ops_per_px_stage_defined": fma_def, "fma_ops_per_px_stage_executed": fma_exe,
        "ex2_per_px_stage_defined": ex2_def, "ex2_per_px_stage_executed": ex2_exe,
        "executed_phi_group_frac": executed_frac,
        "clk_per_px_sm_by_pipe_defined": clk,
        "roofline_value_defined_work": roof_value,
        "x_defined_work_roofline": None if backward else value / world / roof_value,
        "frac_of_measured_ffma": None if backward else achieved / mb["ffma_T_per_s"],
        "xu_frac": None if backward else ex2_exe * px_per_launch / launch_s / 1e12 / xu_peak, "microbench": mb,
        "x_direct_xu_roofline": None if backward else value / world / (xu_peak * 1e12 / EX2_PER_PX_STAGE / 1e6),
        "hbm_gbs_algorithmic": 12.0 * px_per_launch / launch_s / 1e9, "hbm_peak_gbs": read_peaks().get("hbm_gbs"),
        "launch_ms": launch_s * 1e3,
    }
    roofline.update(tensor_extra)
    if use_small:
        roofline.update({"kernel": "small_diffuse_kernel", "achieved": None, "frac": None, "x_defined_work_roofline": None,
                         "formulation": "small-image kernel: all T stages in one launch (cluster of 8 / 16 CTAs per image)",
                         "us_per_call": 1e3 * ms / args.steps,
                         "note": "latency-bound: reported as microseconds per call, not as a roofline fraction (SURVEY.md 8d)"})
    if backward:
        roofline["note"] = "no roofline statement for the joint-training step: its three kernels have no single declared count"
    peak_nominal = xu_peak                               # the opt-in evaluators below are quoted against the XU roofline
    line = {
        "metric": METRIC, "value": value, "unit": "Mpixel-stages/s", "n_gpus": world, "steps": args.steps,
        "warmup": warmup, "ms_per_step": ms / args.steps, "ms_per_step_median": ms_median, "ms_per_step_best": ms_best,
        "higher_is_better": True, "scaling": "strong" if slab else "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": (f"JPEG deblocking TRD^4_7x7 {B}x{H}x{W} (PAPER.md:287), synthetic QCS" if deblock else
                                f"joint-training step (T={T} forward stages + back-propagation, Supp. Eq. 21; dl/du0, dl/dk, "
                                f"dl/dw, dl/dlambda) {B}x{H}x{W} N_k={N_K} {KSIZE}x{KSIZE}; value counts B*H*W*T per step; "
                                f"roofline fields count the forward exponentials only" if backward else
                                f"C{args.workload[1]} {B}x{H}x{W} T={T} N_k={N_K} {KSIZE}x{KSIZE} M=63 "
                                f"(BASELINE.json configs[{int(args.workload[1]) - 1}]), one such batch per GPU"),
                   "global_batch": B if slab else world * B,
                   "parallelism": (f"{world} row slabs of one image, 2rT overlap, no collective" if slab else
                                   f"dp{world} (independent images, no collective)"),
                   "l2": ("inputs larger than L2 (3 planes x %d MB)" % (B * H * W * 4 // 2 ** 20)) if 3 * B * H * W * 4 > 126e6
                   else "working set fits L2 (exploration workload)"},
        "roofline": roofline, "clocks": clocks.summary(),
        "e2e": {"value": e2e_value, "unit": "Mpixel-stages/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps, "matches_device_path": same},
        "gpu_launches": int(launches),
        "paper_context": "GTX 780 Ti: 54.2 Mpixel-stages/s at 3072^2 (PAPER.md:253), other hardware, LUT phi",
    }
    if tile is not None:
        line["tile_kernel"] = {
            "value": tile, "unit": "Mpixel-stages/s", "max_abs_from_default": tile_dist,
            "fma_roofline_frac": N_K * (2 * KSIZE * KSIZE + FACT_GROUPS * FACT_FMA_PER_GROUP) * float(world * B) * H * W * T
                                 * args.steps / (ms_t * 1e-3) / 1e12 / fma_peak,
            "note": "tnrd_set_kernel(2): the same factorised evaluator with both filterings on the FMA pipe (round 1's "
                    "headline kernel, now with dead phi groups skipped); its fraction counts all 8544 defined operations"}
    if win is not None:
        # accounting rule: a variant that skips phi terms reports its executed work against the peak
        # and its throughput as a MULTIPLE of the direct-evaluation XU roofline, never as "% of roofline"
        line["direct_phi"] = {
            "value": direct, "unit": "Mpixel-stages/s", "max_abs_from_default": direct_dist,
            "xu_roofline_frac": EX2_PER_PX_STAGE * float(world * B) * H * W * T * args.steps / (ms_d * 1e-3) / 1e12 / xu_peak,
            "note": "tnrd_set_phi_mode(0): one ex2 per Gaussian (63 per response), bound by the XU pipe: 3024 ex2 per "
                    "pixel-stage against 148 SM x 16/clk x 1.965 GHz"}
        line["windowed_phi"] = {
            "value": win, "unit": "Mpixel-stages/s", "terms_evaluated": 14, "terms_defined": 63,
            "executed_ex2_frac_of_peak": 14 * N_K * float(world * B) * H * W * T * args.steps
                                         / (ms_w * 1e-3) / 1e12 / peak_nominal,
            "x_direct_xu_roofline": win / (peak_nominal * 1e12 / EX2_PER_PX_STAGE / 1e6),
            "note": "tnrd_set_phi_mode(1): 14 of 63 Gaussians per response, dropped terms < 6.7e-10 w each"}
        line["lut_phi"] = {
            "value": lut, "unit": "Mpixel-stages/s", "x_direct_xu_roofline": lut / (peak_nominal * 1e12 / EX2_PER_PX_STAGE / 1e6),
            "max_abs_from_default": lut_dist,
            "note": "tnrd_set_phi_mode(2): 4096-node table + linear interpolation per filter (PAPER.md:572), an approximation"}
    if not args.no_cpu_baseline and world == 1:
        v, cores, sample, _ = oracle_sample(cfg, target_s=args.ref_seconds)
        line["cpu_baseline"] = {"value": v, "unit": "Mpixel-stages/s", "cores": cores, "kind": "oracle",
                                "sample": sample}
        # one thread on the paper's image size and model (C3: 481x321, 48 x 7x7, T = 5), beside the paper's
        # single-thread Matlab row (0.27-0.35 Mpixel-stages/s on a Xeon E5-2680 v2)
        import oracle
        c3 = tnrd_gen.make_config(3)
        nthr = oracle.num_threads()
        oracle.set_num_threads(1)
        try:
            crop = c3["f"][0, 60:260, 140:340]
            t0 = time.perf_counter()
            oracle.diffuse(crop, crop, c3["filters"], c3["rbf_w"], c3["rbf_mu"], c3["rbf_gamma"], c3["lambda"])
            dt1 = time.perf_counter() - t0
        finally:
            oracle.set_num_threads(nthr)
        line["cpu_baseline"]["one_thread_c3"] = {"value": 200 * 200 * c3["T"] / dt1 / 1e6, "unit": "Mpixel-stages/s",
                                                 "sample": f"200x200 crop of the C3 image, T=5, 1 thread, {dt1:.1f} s"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
