#!/usr/bin/env python
"""bench.py — throughput of the hot path (Philox -> RAMBO -> sigmaKin) on B200s.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl reference]

One "step" = one pass of the whole hot path over one batch of synthetic events:
mg_rng -> mg_rambo -> mg_sigmakin (with the event weight), three kernel launches through the C ABI.
Default workload: BASELINE.json configs[4] (g g -> t t~ g g, 2^20 events, FP64), the configuration
north_star's target is quoted on.  Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement".
"""
import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

# name -> (process id, precision, events per step, seed, BASELINE.json config index)
WORKLOADS = {
    "eemumu_16k_fp64": (0, 0, 16384, 42, 0),
    "eemumu_fp64": (0, 0, 1 << 24, 7, 1),
    "eemumu_fp32": (0, 1, 1 << 24, 7, 1),
    "ggtt_fp64": (1, 0, 1 << 22, 7, 2),
    "ggtt_fp32": (1, 1, 1 << 22, 7, 2),
    "ggttg_fp64": (2, 0, 1 << 21, 7, 3),
    "ggttg_fp32": (2, 1, 1 << 21, 7, 3),
    "ggttgg_fp64": (3, 0, 1 << 20, 7, 4),
    "ggttgg_fp32": (3, 1, 1 << 20, 7, 4),
    # quark-initiated channel (not a BASELINE.json configuration: sized like configs[2] / configs[3])
    "qqtt_fp64": (4, 0, 1 << 22, 7, None),
    "qqtt_fp32": (4, 1, 1 << 22, 7, None),
    "qqttg_fp64": (5, 0, 1 << 21, 7, None),
    "qqttg_fp32": (5, 1, 1 << 21, 7, None),
}
PROC_NAME = {0: "e+ e- -> mu+ mu-", 1: "g g -> t t~", 2: "g g -> t t~ g", 3: "g g -> t t~ g g", 4: "u u~ -> t t~", 5: "u u~ -> t t~ g"}
# CPU-baseline sample sizes: about 10-30 s of oracle work on 8 cores
CPU_SAMPLE = {0: 1 << 19, 1: 1 << 19, 2: 1 << 16, 3: 1 << 12, 4: 1 << 17, 5: 1 << 15}
# reference arm: events per step (a bounded sample so that steps+warmup end within minutes)
REF_SAMPLE = {0: 1 << 17, 1: 1 << 17, 2: 1 << 13, 3: 1 << 9, 4: 1 << 15, 5: 1 << 12}
# the kernel bench.py brackets with CUDA events for the roofline (what mg_sigmakin launches for that workload)
KERNEL_NAME = {0: "mg::sigmakin_kernel<mg::Eemumu, %s, false>", 1: "mg::sigmakin_kernel<mg::Ggtt, %s, false>",
               2: "mg::rc::sigmakin_recycle_kernel<mg::RcGgttg, %s, %s, 0>", 3: "mg::rc::sigmakin_recycle_kernel<mg::RcGgttgg, %s, %s, 0>",
               4: "mg::sigmakin_kernel<mg::Qqtt, %s, false>", 5: "mg::sigmakin_kernel<mg::Qqttg, %s, false>"}


def kernel_name(process, prec):
    t = "double" if prec == 0 else "float"
    name = KERNEL_NAME[process]
    return name % ((t, t) if name.count("%s") == 2 else (t,))


PAPER_BASELINE = {"ggttgg_fp64": 5e5, "eemumu_fp64": 1.37e9, "eemumu_fp32": 3.28e9}   # V100

# flop tallies of the shared-memory kernels before the helicity-flip symmetry (commit b02c00b: gen_rc_tables.cuh), (process, precision)
FULL_SUM_FLOPS = {(3, 0): 503313, (3, 1): 498267, (2, 0): 40333, (2, 1): 38435}

# FP64 / FP32 FMA lanes per SM; peak = 148 SMs x lanes x 2 x sm clock
LANES = {0: 64, 1: 128}


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML during the timed region."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.reasons, self.max_mhz = index, False, [], set(), None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                     "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10, "applications_clocks_setting": 0x2}
            while not self.stop_flag:
                self.sm.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
                time.sleep(0.05)
        except Exception as e:       # NVML missing: report that rather than inventing clocks
            self.reasons.add("nvml_unavailable:%s" % type(e).__name__)

    def result(self):
        return {"sm_mhz": statistics.median(self.sm) if self.sm else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons)}


def cpu_baseline(process, seed, sample):
    """The oracle as it stands on the host cores: the whole pipeline (the reported value), and its two legs timed
    separately: Philox + RAMBO (single thread in the oracle's C API) and the matrix element (all threads)."""
    import oracle
    oracle.lib()
    t = time.perf_counter()
    oracle.pipeline(process, seed, 0, sample)
    dt = time.perf_counter() - t
    t = time.perf_counter()
    rho = oracle.uniforms(seed, 0, sample, oracle.N_FINAL[process])
    mom, w, _ = oracle.rambo(rho, oracle.masses(process), 1500.0)
    dt_gen = time.perf_counter() - t
    t = time.perf_counter()
    oracle.me(process, mom)
    dt_me = time.perf_counter() - t
    return {"value": sample / dt, "unit": "MEs/s", "cores": oracle.hardware_threads(), "kind": "oracle",
            "sample": "%d events of %s (Philox -> RAMBO -> ME), oracle FP64, %.1f s" % (sample, PROC_NAME[process], dt),
            "legs": {"rng_rambo_events_per_s": sample / dt_gen, "rng_rambo_threads": 1,
                     "me_events_per_s": sample / dt_me, "me_threads": oracle.hardware_threads()}}


def run_reference(args):
    """The reference arm: the oracle as it stands on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    process, prec, n, seed, cfg = WORKLOADS[args.workload]
    sample = REF_SAMPLE[process]
    oracle.lib()
    for w in range(args.warmup):
        oracle.pipeline(process, seed, w * sample, sample)
    t = time.perf_counter()
    for s in range(args.steps):
        oracle.pipeline(process, seed, (args.warmup + s) * sample, sample)
    dt = time.perf_counter() - t
    value = sample * args.steps / dt
    cores = oracle.hardware_threads()
    desc = "%d events per step of %s, oracle FP64 on %d host threads" % (sample, PROC_NAME[process], cores)
    print(json.dumps({
        "impl": "reference", "metric": "matrix elements/sec", "value": value, "unit": "MEs/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "process": PROC_NAME[process], "events_per_step": sample,
                   "baseline_config": cfg, "note": "bounded sample of the workload"},
        "cpu_baseline": {"value": value, "unit": "MEs/s", "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": "MEs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def time_workload(mg, torch, name, device_index, steps, warmup, dist=None, sampler=None):
    """Times `steps` steps of one workload on this rank.  Returns a dict of measurements."""
    process, prec, n, seed, cfg = WORKLOADS[name]
    P = mg.Process(process, prec, device_index)
    ld = mg.padded_stride(n)
    rnd = P.empty(4 * P.n_final, n, ld)
    mom = P.empty(4 * P.n_external, n, ld)
    w = torch.empty(ld, dtype=P.dtype, device=P.device)
    me = torch.empty(ld, dtype=P.dtype, device=P.device)
    ew = torch.empty(ld, dtype=P.dtype, device=P.device)
    rank = dist.get_rank() if dist else 0
    world = dist.get_world_size() if dist else 1
    # one-off good-helicity filter (A12) on the first events of this rank's range
    P.rng(seed, rank * n, n, out=rnd)
    P.rambo(rnd, n, mom, w)
    mask = P.filter_helicities(mom, 32)

    def step(i):
        first = (i * world + rank) * n          # disjoint global event ranges: weak scaling, no collective
        P.rng(seed, first, n, out=rnd)
        P.rambo(rnd, n, mom, w)
        P.sigmakin(mom, n, me, w, ew)

    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]

    def timed_step(i, k):
        first = (i * world + rank) * n
        P.rng(seed, first, n, out=rnd)
        P.rambo(rnd, n, mom, w)
        ev[k][0].record()
        P.sigmakin(mom, n, me, w, ew)
        ev[k][1].record()

    for i in range(warmup):
        step(i)
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    if sampler:
        sampler.start()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    for k in range(steps):
        timed_step(warmup + k, k)
    t1.record()
    torch.cuda.synchronize()
    if sampler:
        sampler.stop_flag = True
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    total_ms = t0.elapsed_time(t1)
    if dist:
        t = torch.tensor([total_ms], dtype=torch.float64, device=P.device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = t.item()
    kern_ms = statistics.mean(a.elapsed_time(b) for a, b in ev)
    mean_me = me[:n].to(torch.float64).mean().item()
    finite = bool(torch.isfinite(me[:n]).all().item())
    flops = P.flops_per_event(mg.STAGE_SIGMAKIN)
    step_bytes = n * (P.bytes_per_event(mg.STAGE_RNG) + P.bytes_per_event(mg.STAGE_RAMBO) + P.bytes_per_event(mg.STAGE_SIGMAKIN))
    rescued = P.last_rescued() if (prec == 1 and process in (2, 3)) else 0
    return {"P": P, "n": n, "ld": ld, "mask": mask, "total_ms": total_ms, "kern_ms": kern_ms, "mean_me": mean_me, "rescued": rescued,
            "finite": finite, "flops_per_event": flops, "step_bytes": step_bytes, "process": process, "prec": prec,
            "seed": seed, "cfg": cfg, "world": world}


def stage_rates(mg, torch, r, reps=20):
    """A1-A4 alone: HBM GB/s of the RNG, RAMBO and fused generate kernels (north_star: "HBM GB/s for the RNG and RAMBO
    stages"), algorithmic bytes of mg_bytes_per_event over the mean launch time, against MEASURED_PEAKS.json hbm_gbs."""
    P, n, ld = r["P"], r["n"], r["ld"]
    rnd = P.empty(4 * P.n_final, n, ld)
    mom = P.empty(4 * P.n_external, n, ld)
    w = torch.empty(ld, dtype=P.dtype, device=P.device)
    hbm = measured_peaks().get("hbm_gbs")
    calls = {"rng": (lambda i: P.rng(r["seed"], i * n, n, out=rnd), mg.STAGE_RNG),
             "rambo": (lambda i: P.rambo(rnd, n, mom, w), mg.STAGE_RAMBO),
             "generate": (lambda i: P.generate(r["seed"], i * n, n, mom, w), mg.STAGE_GENERATE)}
    me = torch.empty(ld, dtype=P.dtype, device=P.device)
    ew = torch.empty(ld, dtype=P.dtype, device=P.device)
    # A1-A13 in one call, momenta never stored: whole-path MEs/s next to the three-kernel step
    calls["fused_path"] = (lambda i: P.sigmakin_fused(r["seed"], i * n, n, me, w, ew), None)
    # sigmaKin alone, next to its two-kernel form under a CUDA graph: same momenta, same values
    if r["process"] in (2, 3):
        calls["sigmakin"] = (lambda i: P.sigmakin(mom, n, me), None)
        calls["sigmakin_split_graph"] = (lambda i: P.sigmakin_split(mom, n, me=me), None)
    # after the path: batch sums of the event weights and hit-or-miss stream compaction
    fn_f = calls["fused_path"][0]
    fn_f(0)
    es = 8 if r["prec"] == 0 else 4
    wmax = P.weight_sums(ew, n)[2]
    kept = torch.empty(n, dtype=torch.int64, device=P.device)
    nkept = [0]

    d_sums = torch.empty(3, dtype=torch.float64, device=P.device)
    d_cnt = torch.empty(1, dtype=torch.int64, device=P.device)
    nkept[0] = len(P.unweight(r["seed"], 0, ew, n, wmax, kept))
    # device-resident forms (results stay in HBM, no host synchronisation): what a pipeline on the device calls
    calls["weight_sums"] = (lambda i: P.weight_sums_async(ew, n, d_sums), n * es)
    calls["unweight"] = (lambda i: P.unweight_async(r["seed"], 0, ew, n, wmax, kept, d_cnt), n * es + 8 * nkept[0])
    # host-returning forms: the time includes the host round trip
    calls["weight_sums_sync"] = (lambda i: P.weight_sums(ew, n), n * es)
    calls["unweight_sync"] = (lambda i: P.unweight(r["seed"], 0, ew, n, wmax, kept), n * es + 8 * nkept[0])
    out = {}
    for name, (fn, stage) in calls.items():
        for i in range(3):
            fn(i)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record()
        for i in range(reps):
            fn(i)
        b.record()
        torch.cuda.synchronize()
        ms = a.elapsed_time(b) / reps
        if stage is None:
            out[name] = {"ms": ms, "MEs_per_s": n / (ms * 1e-3)}
            continue
        nbytes = stage if name.startswith(("weight_sums", "unweight")) else n * P.bytes_per_event(stage)
        gbs = nbytes / (ms * 1e-3) / 1e9
        out[name] = {"ms": ms, "GB/s": gbs, "frac_hbm": gbs / hbm if hbm else None, "events_per_s": n / (ms * 1e-3)}
        if name.startswith("unweight"):
            out[name].update({"kept": nkept[0], "of": n})
    return out


def small_batch_step(mg, torch, r, reps=200):
    """Config 1 (16 384 events) is launch bound: microseconds per step of (a) the three launches, (b) the same three
    launches replayed from a CUDA graph, (c) the one fused launch (mg_sigmakin_fused)."""
    P, n, ld = r["P"], r["n"], r["ld"]
    rnd = P.empty(4 * P.n_final, n, ld)
    mom = P.empty(4 * P.n_external, n, ld)
    w = torch.empty(ld, dtype=P.dtype, device=P.device)
    me = torch.empty(ld, dtype=P.dtype, device=P.device)
    ew = torch.empty(ld, dtype=P.dtype, device=P.device)

    def three():
        P.rng(r["seed"], 0, n, out=rnd)
        P.rambo(rnd, n, mom, w)
        P.sigmakin(mom, n, me, w, ew)

    def timed(fn):
        for _ in range(5):
            fn()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record()
        for _ in range(reps):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps * 1e3

    out = {"three_launches_us": timed(three), "fused_launch_us": timed(lambda: P.sigmakin_fused(r["seed"], 0, n, me, w, ew))}
    try:
        g = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):
            three()
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=side):
            three()
        out["graph_replay_us"] = timed(g.replay)
    except Exception as e:
        out["graph_replay_us"] = "failed: %s" % e
    out["events"] = n
    return out


def batch_sweep(mg, torch, name, device_index):
    """Throughput against the number of events per launch (PAPER.md:104 Fig. 5 and its two definitions, :156-164:
    kernel only, and kernel + device-to-host copy of the matrix elements)."""
    process, prec, nmax, seed, cfg = WORKLOADS[name]
    P = mg.Process(process, prec, device_index)
    mom, w = P.generate(seed, 0, nmax)
    P.filter_helicities(mom, 32)
    me = torch.empty(mom.shape[1], dtype=P.dtype, device=P.device)
    h_me = torch.empty(nmax, dtype=P.dtype).pin_memory()
    n = 256
    while n <= nmax:
        reps = max(3, min(200, (1 << 22) // n))
        for _ in range(3):
            P.sigmakin(mom, n, me)
        a, b, c = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        torch.cuda.synchronize()
        a.record()
        for _ in range(reps):
            P.sigmakin(mom, n, me)
        b.record()
        for _ in range(reps):
            P.sigmakin(mom, n, me)
            h_me[:n].copy_(me[:n], non_blocking=True)
        c.record()
        torch.cuda.synchronize()
        k_ms, kc_ms = a.elapsed_time(b) / reps, b.elapsed_time(c) / reps
        print(json.dumps({"sweep": name, "events_per_launch": n, "kernel_ms": k_ms, "MEs_per_s_kernel": n / (k_ms * 1e-3),
                          "MEs_per_s_kernel_plus_d2h": n / (kc_ms * 1e-3)}))
        n *= 4


def e2e_measure(mg, torch, r, steps):
    """End to end through the C ABI with HOST buffers: momenta H2D, sigmaKin, ME D2H (mg_sigmakin_host)."""
    P, n, ld = r["P"], r["n"], r["ld"]
    h_mom = torch.empty((4 * P.n_external, ld), dtype=P.dtype).pin_memory()
    h_me = torch.empty(n, dtype=P.dtype).pin_memory()
    h_ref = torch.empty(n, dtype=P.dtype).pin_memory()
    P.run_host(r["seed"], 0, n, h_ref, h_mom)          # fills the pinned host momenta (untimed) and the MEs of one launch
    P.sigmakin_host(h_mom, n, h_me)                    # warm-up
    assert torch.equal(h_me, h_ref), "chunked host call and single launch disagree"
    torch.cuda.synchronize()
    t = time.perf_counter()
    for _ in range(steps):
        P.sigmakin_host(h_mom, n, h_me)
    dt = time.perf_counter() - t
    es = 8 if r["prec"] == 0 else 4
    return {"value": n * steps / dt * r["world"], "unit": "MEs/s", "h2d_bytes_per_step": 4 * P.n_external * ld * es,
            "d2h_bytes_per_step": n * es, "call": "mg_sigmakin_host (pinned host momenta in, host MEs out)"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="ggttgg_fp64", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-extra", action="store_true", help="skip the other workloads and the CPU baseline")
    ap.add_argument("--sweep", action="store_true",
                    help="batch-size sweep of the sigmaKin kernel (PAPER.md:104-108 Fig. 5): one JSON line per size, then exit")
    args = ap.parse_args()
    if args.sweep:
        import torch
        import paper_2106_12631_b200 as mg
        batch_sweep(mg, torch, args.workload, 0)
        return
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
        return

    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # one process per GPU: re-run this command under torchrun (the driver launches it that way itself for N > 1)
        import socket
        sock = socket.socket()
        sock.bind(("127.0.0.1", 0))
        port = sock.getsockname()[1]
        sock.close()
        os.environ.setdefault("NCCL_DEBUG", "INFO")          # the communicator log shows the ranks and the transport
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
                                  "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:])
    import torch
    import paper_2106_12631_b200 as mg
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    if int(os.environ.get("WORLD_SIZE", "1")) != args.gpus:
        raise SystemExit("bench.py --gpus %d was launched with WORLD_SIZE=%s" % (args.gpus, os.environ.get("WORLD_SIZE", "1")))
    dist = None
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    torch.cuda.set_device(local_rank)
    rank = dist.get_rank() if dist else 0

    sampler = ClockSampler(local_rank) if rank == 0 else None
    r = time_workload(mg, torch, args.workload, local_rank, args.steps, args.warmup, dist, sampler)
    if sampler:
        sampler.join(timeout=2)
    e2e = e2e_measure(mg, torch, r, max(2, min(args.steps, 5)))
    if dist:
        t = torch.tensor([e2e["value"] / r["world"]], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MIN)
        e2e["value"] = t.item() * r["world"]

    peaks = measured_peaks()
    sm_max = peaks.get("sm_max_mhz", 1965.0)
    prec = r["prec"]
    peak_tf = 148 * LANES[prec] * 2 * sm_max * 1e6 / 1e12
    n, world = r["n"], r["world"]
    value = n * world * args.steps / (r["total_ms"] * 1e-3)
    achieved_tf = r["flops_per_event"] * n / (r["kern_ms"] * 1e-3) / 1e12
    out = {
        "metric": "matrix elements/sec", "value": value, "unit": "MEs/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": r["total_ms"] / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": (value / world / PAPER_BASELINE[args.workload]) if (args.workload in PAPER_BASELINE and world == 1) else None,
        "dtype": "f64" if prec == 0 else "f32", "data": "synthetic",
        "config": {"workload": args.workload, "process": PROC_NAME[r["process"]], "events_per_step_per_gpu": n,
                   "baseline_config": r["cfg"], "seed": r["seed"], "sqrt_s_gev": 1500.0,
                   "good_helicities": bin(r["mask"]).count("1"), "parallelism": "events sharded, no collective",
                   "l2": "inputs larger than L2: %.0f MB of rnd+momenta traffic per step, new event range every step" % (r["step_bytes"] / 1e6),
                   "paper_baseline": "V100, PAPER.md:116/:159 (context, other hardware)" if args.workload in PAPER_BASELINE else None},
        "e2e": e2e,
        # rng, rambo, sigmaKin per step; FP32 handles of g g -> t t~ g (g) add the double-precision pass over the listed events
        "gpu_launches": (4 if (prec == 1 and r["process"] in (2, 3)) else 3) * args.steps,
        "roofline": {"bound": "alu", "kernel": kernel_name(r["process"], prec), "achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s",
                     "frac": achieved_tf / peak_tf, "traffic": None,
                     "flops_per_event": r["flops_per_event"], "kernel_ms": r["kern_ms"],
                     "peak_kind": "nominal (lanes x clock); the measured_* entries are on-box microbenchmarks of the same pipe",
                     "peak_source": "148 SMs x %d FMA lanes x 2 x %.0f MHz (MEASURED_PEAKS.json sm_max_mhz)" % (LANES[prec], sm_max),
                     # frac counts the flops this kernel EXECUTES.  The QCD kernels use |M(h)|^2 = |M(-h)|^2 (R35): they
                     # evaluate half of the helicity combinations.  For context, the same launch against the flop count of the
                     # same algorithm WITHOUT that symmetry (round-2 kernel before it: 503 313 flop per g g -> t t~ g g event at
                     # 27.4 ms = 0.518 of the peak): not a fraction of executed work, never the headline
                     "flops_per_event_full_helicity_sum": FULL_SUM_FLOPS.get((r["process"], prec)),
                     "frac_vs_full_helicity_sum_flops": (FULL_SUM_FLOPS[(r["process"], prec)] * n / (r["kern_ms"] * 1e-3) / 1e12 / peak_tf)
                     if (r["process"], prec) in FULL_SUM_FLOPS else None},
        "mean_me": r["mean_me"], "all_finite": r["finite"],
    }
    if rank == 0:
        out["clocks"] = sampler.result()
        try:
            from paper_2106_12631_b200 import probe
            out["roofline"]["measured_fma_chain_tflops"] = probe.alu_tflops(prec, local_rank, 0)
            # how the FMA is fed decides its rate on sm_100a: three distinct register operands vs tensor-core FP64
            out["roofline"]["measured_fma_3reg_tflops"] = probe.alu_tflops(prec, local_rank, 1)
            if prec == 0:
                out["roofline"]["measured_dmma_tflops"] = probe.alu_tflops(prec, local_rank, 2)
        except Exception as e:
            out["roofline"]["measured_fma_chain_tflops"] = "failed: %s" % e
        try:
            out["stages"] = stage_rates(mg, torch, r)
        except Exception as e:
            out["stages"] = "failed: %s" % e
        # DRAM bytes per launch of that kernel from a committed ncu --set full capture of this workload, if there is one
        tr = os.path.join(ROOT, "profiles", "traffic.json.txt")
        ent = json.load(open(tr)).get(args.workload) if os.path.exists(tr) else None
        if isinstance(ent, dict):
            out["roofline"]["traffic"] = ent.get("bytes")
            out["roofline"]["traffic_source"] = ent.get("source")
        else:
            out["roofline"]["traffic_source"] = "no ncu capture of this workload under profiles/"
        if prec == 1 and r["process"] in (2, 3):
            out["config"]["fp32_events_recomputed_in_double"] = r["rescued"]
    if rank == 0 and world == 1 and not args.no_extra:
        out["cpu_baseline"] = cpu_baseline(r["process"], r["seed"], CPU_SAMPLE[r["process"]])
        others = []
        for name in sorted(WORKLOADS):
            if name == args.workload:
                continue
            try:
                o = time_workload(mg, torch, name, local_rank, 3, 3)
                pk = 148 * LANES[o["prec"]] * 2 * sm_max * 1e6 / 1e12
                tf = o["flops_per_event"] * o["n"] / (o["kern_ms"] * 1e-3) / 1e12
                others.append({"workload": name, "value": o["n"] * 3 / (o["total_ms"] * 1e-3), "unit": "MEs/s",
                               "sigmakin_MEs_per_s": o["n"] / (o["kern_ms"] * 1e-3), "sigmakin_ms": o["kern_ms"],
                               "kernel": kernel_name(o["process"], o["prec"]),
                               "alu_frac_of_nominal": tf / pk, "flops_per_event": o["flops_per_event"],
                               # the same launch against the HBM roofline: momenta read, ME / weights written (mg_bytes_per_event)
                               "sigmakin_hbm_frac": (o["n"] * o["P"].bytes_per_event(mg.STAGE_SIGMAKIN) / (o["kern_ms"] * 1e-3) / 1e9 / peaks["hbm_gbs"]) if peaks.get("hbm_gbs") else None,
                               "mean_me": o["mean_me"],
                               "all_finite": o["finite"], "stages": stage_rates(mg, torch, o, reps=10)})
                if o["prec"] == 1 and o["process"] in (2, 3):
                    others[-1]["fp32_events_recomputed_in_double"] = o["rescued"]
                if name == "eemumu_16k_fp64":
                    others[-1]["small_batch"] = small_batch_step(mg, torch, o)
                del o
                torch.cuda.empty_cache()
            except Exception as e:
                others.append({"workload": name, "error": str(e)})
        out["other_workloads"] = others
    if rank == 0:
        print(json.dumps(out))
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
