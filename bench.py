#!/usr/bin/env python
"""bench.py -- CKKS HE-mult + relinearise + rescale throughput at N = 2^16, logQ = 1240 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

One "step" = one pass of the whole hot path (decompose, forward NTT, tensor pointwise,
inverse NTT, CRT + mod Q, relinearise with evk mod PQ + divide by P, rescale by 2^40) over one batch of 4
synthetic ciphertext pairs per GPU (BASELINE.json configs[4]).  Prints ONE JSON line (rank 0).
Multi-GPU: the batch dimension shards with no data-path collective -> weak scaling, evk replicated.
`--impl reference` times the CPU oracle (oracle/, test infrastructure) on a bounded sample (one ring product of the
workload's shape per step, mod Q and mod PQ in the 4 : 2 mix of an op) on the host cores.
`python bench.py --gpus N` without a launcher re-executes itself under torch.distributed.run with N ranks.
`--sweep`: the standalone polymul sweep; `--table1`: the operations of the paper's Table 1 at the paper's own shape
(cnum = 4, N = 2^16, logQ = 1024), one JSON line each with the paper's T4 latency beside it (context, not a target);
`--configs`: the call of each of the five BASELINE.json configs, one JSON line each.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "CKKS HE-mult+relin+rescale ops/s at N=2^16 logQ=1240"
UNIT = "ops/s"
WORKLOADS = {
    # name: (N, logQ, logP, batch, rescale bits)
    "c5": (1 << 16, 1240, 1240, 4, 40),      # BASELINE.json configs[4], the configuration the metric is quoted on
    "c3": (1 << 15, 620, 620, 8, 40),
    "c1": (1 << 10, 128, 128, 1, 40),
}
# DRAM bytes per launch of each kernel class come from a committed `ncu --set full` capture of this same command
# (profiles/dram_traffic.csv: class, launches per step, dram__bytes_read.sum + dram__bytes_write.sum per launch, the sha256
# of the kernel sources the capture was taken with, the capture's file name).  A capture taken with other kernel sources
# than the ones that are running is refused: `traffic` is then null and `traffic_source` says why.
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "dram_traffic.csv")
CSRC = os.path.join(ROOT, "paper_2607_05920_b200", "csrc")


def kernel_source_hash() -> str:
    import hashlib
    h = hashlib.sha256()
    for name in sorted(os.listdir(CSRC)):
        if name.endswith((".cu", ".cuh", ".hpp")):
            with open(os.path.join(CSRC, name), "rb") as f:
                h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()[:16]


def committed_traffic(kernel_class: str):
    """(bytes per launch or None, source string) for one kernel class from profiles/dram_traffic.csv."""
    try:
        with open(TRAFFIC_CSV) as f:
            rows = [r.strip().split(",") for r in f if r.strip() and not r.startswith("#")]
    except OSError:
        return None, "no committed capture (profiles/dram_traffic.csv missing)"
    head = kernel_source_hash()
    for r in rows[1:]:
        if len(r) >= 5 and r[0] == kernel_class:
            if r[3] != head:
                return None, f"stale: {r[4]} was captured with kernel sources {r[3]}, running {head}"
            return float(r[2]), f"{r[4]} (ncu --set full, same command, kernel sources {r[3]})"
    return None, f"no row for {kernel_class} in profiles/dram_traffic.csv"


def workload_string(name: str) -> str:
    N, logQ, logP, B, p_bits = WORKLOADS[name]
    tag = " (BASELINE.json configs[4])" if name == "c5" else ""
    return f"{name}: CKKS N={N} logQ={logQ} logP={logP} batch={B}/GPU rescale={p_bits}{tag}"


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured"
    except Exception:
        return 6650.0, "fallback"


# ---- algorithmic work model of the algorithm actually shipped ---------------------------------------------
def work_model(N, logQ, logP, L, L_PQ, K1, K2, B):
    """Per kernel class and step (B ops): NTT butterflies, other multiplier-pipe work in units of one mad.lo.u32
    (a mul.hi / mul.wide issues at half that rate on B200 and counts 2), and the HBM bytes if every intermediate makes
    exactly one round trip.  The base-conversion contractions run on the tensor cores and are not counted here."""
    logN = N.bit_length() - 1
    half = N // 2
    fwd_t, inv_t = 4 * K1 + K2, 3 * K1 + 2 * K2          # transforms per op
    bf = {
        "decompose": 0,
        "ntt_fwd": B * fwd_t * half * (logN - 8),           # forward column pass
        "pointwise": B * (fwd_t + inv_t) * half * 8,        # fused rows: last forward + first inverse pass
        "ntt_inv": B * inv_t * half * (logN - 8),           # inverse column pass
        "crt": 0, "rescale": 0,
    }
    units = {
        "decompose": B * N * fwd_t * 3,                      # per residue: mul.hi (2) + mul.lo (1) of the Barrett step
        "ntt_fwd": 0,
        "pointwise": B * N * (K1 * 17 + K2 * 10),            # tensor: 4 wide products + 3 reductions; relin: 2 + 2
        "ntt_inv": B * N * inv_t * 4,                        # final Shoup multiplication by the folded constant
        "crt": B * N * (3 * L + 2 * L_PQ) * 8,               # per limb of V: four 32 x 32 -> 64 multiply-adds
        "rescale": 0,
    }
    w = 4
    byt = {   # bytes each class must move if every intermediate makes exactly one HBM round trip
        "decompose": B * N * w * (4 * L + L + 4 * K1 + K2),
        "ntt_fwd": B * N * w * 2 * fwd_t,                                  # forward column pass, in place
        "pointwise": B * N * w * (4 * K1 + 3 * K1 + K2 + 2 * K2 + 2 * K2),  # fused rows: operands in, products out, evk-hat per item
        "ntt_inv": B * N * w * 2 * inv_t,                                  # inverse column pass, in place
        "crt": B * N * w * (3 * K1 + 3 * L + 2 * K2 + 2 * L + 2 * L),
        "rescale": 0,
    }
    compulsory = B * N * w * (4 * L + 2 * L) + N * w * 2 * K2      # read 2 cts, write 1, evk-hat once per batch
    return bf, units, byt, compulsory


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line).  nvidia-smi needs a
    few hundred milliseconds to start, so the sampler is started before the warm-up, waited on until its first line
    is there, and only the samples whose timestamps fall inside [mark_start(), mark_end()] are kept."""

    FIELDS = ("timestamp,index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
              "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.proc = None
        self.t0 = self.t1 = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + self.FIELDS, "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=self.tmp, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None
            return
        deadline = time.time() + 3.0
        while time.time() < deadline and os.path.getsize(self.tmp.name) == 0:
            time.sleep(0.02)

    def mark_start(self):
        self.t0 = time.time()

    def mark_end(self):
        self.t1 = time.time()

    def stop(self):
        import datetime
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is not None:
            time.sleep(0.05)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()
        try:
            self.tmp.flush()
            with open(self.tmp.name) as f:
                rows = [r.strip().split(", ") for r in f if r.strip()]
            os.unlink(self.tmp.name)
            rows = [r for r in rows if len(r) >= 10]
            keep = []
            for r in rows:
                try:
                    ts = datetime.datetime.strptime(r[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                except Exception:
                    continue
                if self.t0 is not None and self.t1 is not None and self.t0 - 0.02 <= ts <= self.t1 + 0.02:
                    keep.append(r)
            out["samples_total"] = len(rows)
            if not keep:            # region shorter than the sampling period: fall back to the samples around it
                keep = rows[-3:]
            sm = sorted(float(r[2]) for r in keep)
            if sm:
                out["sm_mhz"] = sm[len(sm) // 2]
                out["sm_max_mhz"] = float(keep[0][3])
                out["samples"] = len(sm)
                names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
                seen = set()
                for r in keep:
                    for name, val in zip(names, r[6:10]):
                        if val.strip().lower().startswith("active"):
                            seen.add(name)
                out["reasons"] = sorted(seen)
        except Exception:
            pass
        return out


# ---- distributed plumbing (also exercised on CPU with gloo in tests/test_bench_dist.py) ---------------------------------
def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def dist_init(backend: str):
    import torch.distributed as dist
    rank, _, world = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world


def barrier(world: int):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(x: float, world: int, device="cpu") -> float:
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def shard_units(per_gpu_batch: int, world: int):
    """Weak scaling: every rank owns `per_gpu_batch` independent ciphertext pairs; total = world * per_gpu_batch."""
    return per_gpu_batch, per_gpu_batch * world


# ---- the CPU oracle arm ---------------------------------------------------------------------------------------------------
# One op on the oracle = 4 ring products mod Q (the tensor product) + 2 mod PQ (the key switch); the divide-by-P, the
# additions and the rescale are a fraction of a percent beside them.  Both kinds of product are timed in the run.
def oracle_sample_product(N, logQ, logP=0, seed=0):
    """Time ONE ring product of the workload's shape on the oracle (its own NTT route): a (< Q) times b (< Q when
    logP == 0: a tensor-product term; < PQ = 2^(logP + logQ) else: a key-switch term, reduced mod PQ).  Seconds."""
    import synth
    from oracle import ring
    from oracle.limbs import from_limbs
    g = synth.rng(seed)
    a = from_limbs(synth.uniform_limbs(g, (), N, logQ))
    b = from_limbs(synth.uniform_limbs(g, (), N, logQ + logP))
    t0 = time.perf_counter()
    ring.pm(a, b, 1 << (logQ + logP))
    return time.perf_counter() - t0


def oracle_ops_per_s(t_q: float, t_pq: float) -> float:
    return 1.0 / (4.0 * t_q + 2.0 * t_pq)


def run_reference(args):
    """The oracle as it stands on the host cores: at this size its ring product goes through its own NTT route
    (oracle.ring.pm).  A step times ONE ring product of one pair of the workload's shape -- mod Q in two steps out of three,
    mod PQ in the third, the 4 : 2 mix of an op -- and the line converts the two measured means to ops/s."""
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    N, logQ, logP, B, p_bits = WORKLOADS[args.workload]
    for i in range(args.warmup):
        oracle_sample_product(N, logQ, logP if i % 3 == 2 else 0, seed=100 + i)
    tq, tpq = [], []
    t0 = time.perf_counter()
    for i in range(args.steps):
        if i % 3 == 2:
            tpq.append(oracle_sample_product(N, logQ, logP, seed=i))
        else:
            tq.append(oracle_sample_product(N, logQ, 0, seed=i))
    dt = time.perf_counter() - t0
    t_q = sum(tq) / len(tq)
    t_pq = sum(tpq) / len(tpq) if tpq else 2.0 * t_q          # fewer than three steps: no mod-PQ sample, assume twice
    value = oracle_ops_per_s(t_q, t_pq)
    sample = (f"per step 1 ring product of 1 pair (oracle.ring.pm, own NTT route): {len(tq)} mod Q = {t_q:.1f} s each, "
              f"{len(tpq)} mod PQ = {t_pq:.1f} s each; an op = 4 mod Q + 2 mod PQ = {4 * t_q + 2 * t_pq:.1f} s")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int (python big integers, numpy uint64 NTT)", "data": "synthetic",
        "config": {"workload": workload_string(args.workload)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle (python, 1 core, extrapolated from single ring products)",
                         "host_cores": os.cpu_count(), "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)
    return 0


# ---- the CUDA arm -----------------------------------------------------------------------------------------------------------
def run_ours(args):
    import numpy as np
    import torch
    import synth
    import paper_2607_05920_b200 as fhe

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback on the product path)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist_init("nccl")
    N, logQ, logP, B, p_bits = WORKLOADS[args.workload]
    ctx = fhe.Context(N, logQ, logP)
    g = synth.rng(1000 + rank)

    def dev_limbs(lead, bits):
        a = synth.uniform_limbs(g, lead, N, bits)
        return torch.from_numpy(a.view(np.int32)).to(dev)

    ct1, ct2 = dev_limbs((B, 2), logQ), dev_limbs((B, 2), logQ)
    ctx.fhe_set_evk(dev_limbs((2,), logQ + logP))
    out = torch.empty((B, 2, ctx.L, N), dtype=torch.int32, device=dev)
    stream = torch.cuda.current_stream(dev)

    def step():
        ctx.fhe_mult_relin_rescale(ct1, ct2, p_bits, out=out, stream=stream)

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    sampler.mark_start()
    # ---- timed region: K steps, device time on the launching stream, max over ranks ----
    l0 = ctx.launch_count()
    barrier(world)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    torch.cuda.synchronize()
    barrier(world)
    ms_total = max_over_ranks(e0.elapsed_time(e1), world, dev)
    launches = ctx.launch_count() - l0
    _, total_units = shard_units(B, world)
    value = total_units * args.steps / (ms_total / 1e3)

    # ---- per-kernel durations over an instrumented repeat of the region (event pair around every launch) ----
    ctx.fhe_debug_timing(True)
    torch.cuda.synchronize()
    s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s0.record(stream)
    for _ in range(args.steps):
        step()
    s1.record(stream)
    torch.cuda.synchronize()
    per_class = ctx.fhe_debug_timing_read()
    ms_instr = s0.elapsed_time(s1)
    ctx.fhe_debug_timing(False)

    # ---- the same K steps replayed from ONE CUDA graph (the calls allocate nothing and never synchronise, so a step
    # captures as it is, programmatic-dependent-launch edges included): what the launch overhead of 12 kernels costs ----
    graph_info = {"ms_per_step": None}
    try:
        side = torch.cuda.Stream(dev)
        side.wait_stream(stream)
        with torch.cuda.stream(side):
            ctx.fhe_mult_relin_rescale(ct1, ct2, p_bits, out=out, stream=side)
        side.synchronize()
        cg = torch.cuda.CUDAGraph()
        with torch.cuda.graph(cg, stream=side):
            ctx.fhe_mult_relin_rescale(ct1, ct2, p_bits, out=out, stream=torch.cuda.current_stream(dev))
        for _ in range(3):
            cg.replay()
        torch.cuda.synchronize()
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record(stream)
        for _ in range(args.steps):
            cg.replay()
        g1.record(stream)
        torch.cuda.synchronize()
        graph_info = {"ms_per_step": g0.elapsed_time(g1) / args.steps, "what": "one captured step (12 launches) replayed with cudaGraphLaunch"}
    except Exception as ex:                                        # a driver that refuses the capture: report, do not hide the main line
        graph_info = {"ms_per_step": None, "error": str(ex)[:200]}

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ----
    h1, h2 = ct1.cpu().pin_memory(), ct2.cpu().pin_memory()
    hout = torch.empty((B, 2, ctx.L, N), dtype=torch.int32).pin_memory()
    ctx.fhe_mult_relin_rescale_host(h1, h2, p_bits, h_out=hout, stream=stream)
    same = bool(torch.equal(hout, out.cpu()))
    barrier(world)
    torch.cuda.synchronize()
    e2e_steps = max(3, min(args.steps, 10))
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        ctx.fhe_mult_relin_rescale_host(h1, h2, p_bits, h_out=hout, stream=stream)   # synchronises the stream itself
    e2e_ms = max_over_ranks((time.perf_counter() - t0) * 1e3, world, dev)
    e2e_value = total_units * e2e_steps / (e2e_ms / 1e3)
    sampler.mark_end()       # the timed, the instrumented and the end-to-end steps: all of them the same load
    clocks = sampler.stop() if rank == 0 else None
    ct_bytes = B * 2 * ctx.L * N * 4

    if rank != 0:
        return 0
    hbm_gbs, peak_kind = _peaks()
    bf, units, byt, compulsory = work_model(N, logQ, logP, ctx.L, ctx.L_PQ, ctx.K1, ctx.K2, B)
    # integer peaks measured in this run, register-only (fhe_debug_int_peak): the NTT butterfly as the kernels execute
    # it, and mad.lo.u32 for the remaining multiplier-pipe work
    bf_peak, mad_peak, mulhi_peak = (ctx.fhe_debug_int_peak(m) for m in (0, 1, 2))

    def t_int(k):
        return bf[k] / bf_peak + units[k] / mad_peak

    kern = {k: {"ms_per_step": v[0] / args.steps, "launches_per_step": v[1] / args.steps,
                "share": v[0] / max(1e-9, sum(x[0] for x in per_class.values())),
                "gbutterfly_per_step": bf[k] / 1e9, "gmulunit_per_step": units[k] / 1e9, "mb_per_step": byt[k] / 1e6,
                "t_int_ms": t_int(k) * 1e3, "t_hbm_ms": byt[k] / (hbm_gbs * 1e9) * 1e3} for k, v in per_class.items()}
    top = max(per_class, key=lambda k: per_class[k][0])
    n_launch_top = max(1, per_class[top][1])
    avg_launch_s = per_class[top][0] / 1e3 / n_launch_top
    t_hbm = byt[top] / (hbm_gbs * 1e9)
    # a second, mix-independent integer ceiling for the butterfly: one mul.hi and two mad.lo per butterfly at the measured
    # instruction rates -- it cannot move when the kernels' own butterfly code changes
    bf_peak_instr = 1.0 / (1.0 / mulhi_peak + 2.0 / mad_peak)
    if t_int(top) >= t_hbm and bf[top] > 0:
        ach = bf[top] * args.steps / n_launch_top / avg_launch_s
        roof = {"bound": "alu", "kernel": top, "achieved": ach / 1e9, "peak": bf_peak / 1e9, "unit": "Gbutterfly/s",
                "peak_kind": "measured in this run: the kernels' own forward butterfly, register-only (fhe_debug_int_peak; DESIGN.md 7)",
                "frac_vs_instruction_peak": ach / bf_peak_instr, "instruction_peak": bf_peak_instr / 1e9,
                "instruction_peak_kind": "1 mul.hi.u32 + 2 mad.lo.u32 per butterfly at the rates measured in this run"}
    else:
        roof = {"bound": "hbm", "kernel": top, "achieved": byt[top] * args.steps / n_launch_top / avg_launch_s / 1e9,
                "peak": hbm_gbs, "unit": "GB/s", "peak_kind": peak_kind}
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["traffic"], roof["traffic_source"] = committed_traffic(top) if args.workload == "c5" else (None, "captures exist for c5 only")
    roof["algorithmic_bytes_per_launch"] = byt[top] * args.steps / n_launch_top
    roof["avg_launch_ms"] = avg_launch_s * 1e3
    roof["hbm_frac"] = byt[top] * args.steps / n_launch_top / avg_launch_s / 1e9 / hbm_gbs
    # whole-path roofline (north_star): slower of the integer work at the measured integer peaks and the compulsory
    # bytes at the measured HBM bandwidth
    t_path_alu = sum(t_int(k) for k in bf)
    t_path_hbm = compulsory / (hbm_gbs * 1e9)
    t_step = ms_total / args.steps / 1e3
    path = {"t_int_ms": t_path_alu * 1e3, "t_hbm_ms": t_path_hbm * 1e3, "t_measured_ms": t_step * 1e3,
            "frac": max(t_path_alu, t_path_hbm) / t_step, "gbutterfly_per_step": sum(bf.values()) / 1e9,
            "compulsory_mb_per_step": compulsory / 1e6,
            "frac_vs_instruction_peak": max(sum(bf[k] / bf_peak_instr + units[k] / mad_peak for k in bf), t_path_hbm) / t_step,
            "int_peaks": {"gbutterfly_per_s": bf_peak / 1e9, "gbutterfly_per_s_from_instruction_rates": bf_peak_instr / 1e9,
                          "gmadlo_per_s": mad_peak / 1e9, "gmulhi_per_s": mulhi_peak / 1e9}}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        t_q, t_pq = oracle_sample_product(N, logQ, 0), oracle_sample_product(N, logQ, logP)
        cpu = {"value": oracle_ops_per_s(t_q, t_pq), "unit": UNIT, "cores": 1,
               "kind": "oracle (python, 1 core, extrapolated from single ring products)", "host_cores": os.cpu_count(),
               "sample": (f"1 ring product mod Q ({t_q:.1f} s) and 1 mod PQ ({t_pq:.1f} s) of 1 pair (oracle.ring.pm, own NTT "
                          f"route), both timed in this run; an op = 4 mod Q + 2 mod PQ = {4 * t_q + 2 * t_pq:.1f} s")}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u32 (exact integer)", "data": "synthetic",
        "config": {"workload": workload_string(args.workload),
                   "L": ctx.L, "K1": ctx.K1, "K2": ctx.K2, "global_batch": total_units, "parallelism": f"batch-sharded x{world}, no collective",
                   "l2": "inputs + workspace per step (~0.9 GB) exceed the 126 MB L2; no explicit flush"},
        "clocks": clocks, "gpu_launches": int(launches),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 2 * ct_bytes, "d2h_bytes_per_step": ct_bytes,
                "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps, "matches_device_result": same},
        "roofline": roof, "path_roofline": path, "kernels": kern,
        "instrumented_ms_per_step": ms_instr / args.steps,
        "cpu_baseline": cpu,
        "latency_us_per_op": ms_total / args.steps / B * 1e3,
        "cuda_graph": graph_info,
    }
    print(json.dumps(line), flush=True)
    return 0


# ---- the standalone polymul sweep (BASELINE.json configs[4]): not part of the default line ----------------
def run_sweep(args):
    import numpy as np
    import torch
    import synth
    import paper_2607_05920_b200 as fhe

    rank, local_rank, world = dist_env()
    if rank != 0:
        return 0
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    hbm_gbs, _ = _peaks()
    stream = torch.cuda.current_stream(dev)
    # NEXT-1 streaming kernels at the C5 shape: a batch of 64 ciphertexts (2.6 GB of traffic per call), against HBM
    ctx = fhe.Context(1 << 16, 1240, 1240)
    g = synth.rng(0)
    x1 = torch.from_numpy(synth.uniform_limbs(g, (1, 2), 1 << 16, 1240).view(np.int32)).to(dev).expand(64, 2, ctx.L, 1 << 16).contiguous()
    x2 = x1.clone()
    y = torch.empty_like(x1)
    pt = x2[:, 0].contiguous()                                   # one plaintext polynomial per ciphertext
    for name, fn, nbuf in (("fhe_add", lambda: ctx.fhe_add(x1, x2, out=y), 3), ("fhe_sub", lambda: ctx.fhe_sub(x1, x2, out=y), 3),
                           ("fhe_negate", lambda: ctx.fhe_negate(x1, out=y), 2), ("fhe_moddown", lambda: ctx.fhe_moddown(x1, 1200, out=y), 2),
                           ("fhe_mult_scalar", lambda: ctx.fhe_mult_scalar(x1, -12345, out=y), 2),
                           ("fhe_add_plain", lambda: ctx.fhe_add_plain(x1, pt, 1, out=y), 2.5)):
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(5):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 5
        byts = nbuf * x1.numel() * 4
        print(json.dumps({"sweep": True, "metric": name + " ciphertexts/s", "value": 64 / (ms / 1e3), "unit": "ciphertexts/s",
                          "N": 1 << 16, "logQ": 1240, "batch": 64, "ms_per_call": ms, "gb_per_s": byts / (ms / 1e3) / 1e9,
                          "roofline": {"bound": "hbm", "achieved": byts / (ms / 1e3) / 1e9, "peak": hbm_gbs, "unit": "GB/s",
                                       "frac": byts / (ms / 1e3) / 1e9 / hbm_gbs}, "data": "synthetic"}), flush=True)
    # NEXT-2: rotation (automorphism + key switch with a rotation key) of a batch of 4 ciphertexts at the C5 shape
    ctx.fhe_set_rotation_key(0, 5, torch.from_numpy(synth.uniform_limbs(g, (2,), 1 << 16, 2480).view(np.int32)).to(dev))
    xr = x1[:4].contiguous()
    yr = torch.empty_like(xr)
    for _ in range(3):
        ctx.fhe_rotate(xr, 0, out=yr, stream=stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(10):
        ctx.fhe_rotate(xr, 0, out=yr, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / 10
    print(json.dumps({"sweep": True, "metric": "fhe_rotate ciphertexts/s", "value": 4 / (ms / 1e3), "unit": "ciphertexts/s",
                      "N": 1 << 16, "logQ": 1240, "logP": 1240, "batch": 4, "ms_per_call": ms, "data": "synthetic"}), flush=True)
    del ctx, x1, x2, y, xr, yr
    torch.cuda.empty_cache()
    for logN in (12, 13, 14, 15, 16):
        for logQ in (64, 256, 620, 1240, 2480):
            N = 1 << logN
            ctx = fhe.Context(N, logQ, 32)
            L, K = ctx.L, ctx.K_pm
            batch = max(1, round(2e9 / (2 * N * L * 4)))           # about 2 GB of operands
            g = synth.rng(0)
            # one seeded pair, repeated: the kernels have no data-dependent control flow
            a1 = torch.from_numpy(synth.uniform_limbs(g, (1,), N, logQ).view(np.int32)).to(dev)
            b1 = torch.from_numpy(synth.uniform_limbs(g, (1,), N, logQ).view(np.int32)).to(dev)
            a = a1.expand(batch, L, N).contiguous()
            b = b1.expand(batch, L, N).contiguous()
            out = torch.empty_like(a)
            for _ in range(2):
                ctx.fhe_polymul(a, b, out=out, stream=stream)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            reps = max(3, args.steps // 4)
            e0.record(stream)
            for _ in range(reps):
                ctx.fhe_polymul(a, b, out=out, stream=stream)
            e1.record(stream)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / reps
            w = 4
            # algorithmic bytes of the plan this cell runs: decompose a, b | transforms and products | CRT.  N = 2^12 runs the
            # transforms in one kernel (operands in, product out: 3K words per point), the other N in three passes (9K)
            ntt_words = 3 * K if N == (1 << 12) else (2 * 2 * K + 2 * K + K + 2 * K)
            alg = batch * N * w * (2 * L + 2 * K) + batch * N * w * ntt_words + batch * N * w * (K + L)
            cpu = None
            if N <= (1 << 14) and not args.no_cpu_baseline:
                # the oracle beside it: one pair per cell, cells with N <= 2^14 only, one host core
                from oracle import ring
                from oracle.limbs import from_limbs
                ha, hb = from_limbs(a1[0].cpu().numpy().view(np.uint32)), from_limbs(b1[0].cpu().numpy().view(np.uint32))
                t0 = time.perf_counter()
                ring.pm(ha, hb, 1 << logQ)
                t_or = time.perf_counter() - t0
                cpu = {"value": 1.0 / t_or, "unit": "polymuls/s", "cores": 1, "kind": "oracle", "host_cores": os.cpu_count(),
                       "sample": f"1 pair of this cell (oracle.ring.pm) = {t_or:.2f} s; cells with N <= 2^14 only"}
            print(json.dumps({"sweep": True, "metric": "polymuls/s", "value": batch / (ms / 1e3), "unit": "polymuls/s",
                              "N": N, "logQ": logQ, "L": L, "K": K, "batch": batch, "ms_per_call": ms,
                              "us_per_polymul": ms * 1e3 / batch, "algorithmic_gb_per_s": alg / (ms / 1e3) / 1e9,
                              "hbm_frac_of_plan": alg / (ms / 1e3) / 1e9 / hbm_gbs, "dtype": "u32 (exact integer)",
                              "data": "synthetic", "cpu_baseline": cpu}), flush=True)
            del ctx, a, b, out
            torch.cuda.empty_cache()
    return 0


# ---- the paper's Table 1, at the paper's own workload shape: context beside the T4 figures ------------
# cnum = 4 ciphertexts per CipherTensor, logN = 16, logQ = 1024, logp = 60; the evaluation / rotation keys
# are taken mod P Q with logP = logQ (the HEAAN Q^2 key is that case, A2).  One JSON line per operation this
# library has (13 of the 14 rows: bootstrapping is a circuit the paper does not describe), each with the
# paper's T4 latency next to it.  Inputs are uniform random limbs (as the paper's "random ciphertexts"); four input / output
# sets are cycled so that the working set (> 500 MB) exceeds the 126 MB L2.
PAPER_TABLE1_T4_S = {   # operation -> (CipherTensor latency in seconds on a Tesla T4, PAPER.md line)
    "negate_pairwise_into": (0.0191, 766), "moddownBy_pairwise_into": (0.0131, 767), "rescaleBy_pairwise_into": (0.0770, 768),
    "conjugate_pairwise_into": (5.5614, 769), "mult_pairwise_into": (8.1862, 770), "leftrotate_broadcast_into": (5.6852, 771),
    "add_pairwise_into": (0.0286, 772), "sub_pairwise_into": (0.0260, 773), "addconst_broadcast_into": (0.0007, 774),
    "addconst_pairwise_into": (0.0170, 775), "imult_pairwise_into": (0.0170, 776), "multconst_broadcast_into": (0.6219, 777),
    "multconstvec_pairwise_into": (1.9930, 778),
}


def run_table1(args):
    import numpy as np
    import torch
    import synth
    import paper_2607_05920_b200 as fhe

    rank, local_rank, world = dist_env()
    if rank != 0:
        return 0
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    stream = torch.cuda.current_stream(dev)
    N, logQ, logP, B, p_bits, NSET = 1 << 16, 1024, 1024, 4, 60, 4
    ctx = fhe.Context(N, logQ, logP)
    g = synth.rng(2024)

    def limbs(lead, bits):
        return torch.from_numpy(synth.uniform_limbs(g, lead, N, bits).view(np.int32)).to(dev)

    xs = [limbs((B, 2), logQ) for _ in range(NSET)]
    ys = [limbs((B, 2), logQ) for _ in range(NSET)]
    pts = [limbs((B,), logQ) for _ in range(NSET)]
    outs = [torch.empty_like(xs[0]) for _ in range(NSET)]
    out3 = [torch.empty((B, 3, ctx.L, N), dtype=torch.int32, device=dev) for _ in range(NSET)]
    ctx.fhe_set_evk(limbs((2,), logQ + logP))
    ctx.fhe_set_rotation_key(0, 5, limbs((2,), logQ + logP))             # rotation by one slot: X -> X^5
    ctx.fhe_set_rotation_key(1, 2 * N - 1, limbs((2,), logQ + logP))     # conjugation: X -> X^-1

    def mult(i):
        ctx.fhe_he_mult(xs[i], ys[i], out=out3[i], stream=stream)
        ctx.fhe_relinearize(out3[i], out=outs[i], stream=stream)

    ops = (   # paper's name, the call, what it is here
        ("negate_pairwise_into", lambda i: ctx.fhe_negate(xs[i], out=outs[i]), "fhe_negate"),
        ("moddownBy_pairwise_into", lambda i: ctx.fhe_moddown(xs[i], logQ - p_bits, out=outs[i]), "fhe_moddown to logq = 964"),
        ("rescaleBy_pairwise_into", lambda i: ctx.fhe_rescale(xs[i], p_bits, out=outs[i], stream=stream), "fhe_rescale by 2^60"),
        ("conjugate_pairwise_into", lambda i: ctx.fhe_rotate(xs[i], 1, out=outs[i], stream=stream), "fhe_rotate, key for X -> X^(2N-1)"),
        ("mult_pairwise_into", mult, "fhe_he_mult + fhe_relinearize"),
        ("leftrotate_broadcast_into", lambda i: ctx.fhe_rotate(xs[i], 0, out=outs[i], stream=stream), "fhe_rotate, key for X -> X^5"),
        ("add_pairwise_into", lambda i: ctx.fhe_add(xs[i], ys[i], out=outs[i]), "fhe_add"),
        ("sub_pairwise_into", lambda i: ctx.fhe_sub(xs[i], ys[i], out=outs[i]), "fhe_sub"),
        ("addconst_broadcast_into", lambda i: ctx.fhe_add_plain(xs[i], pts[i][:1], B, out=outs[i]), "fhe_add_plain, one plaintext for the batch"),
        ("addconst_pairwise_into", lambda i: ctx.fhe_add_plain(xs[i], pts[i], 1, out=outs[i]), "fhe_add_plain, one plaintext per ciphertext"),
        ("imult_pairwise_into", lambda i: ctx.fhe_mul_monomial(xs[i], N // 2, out=outs[i]), "fhe_mul_monomial by X^(N/2)"),
        ("multconst_broadcast_into", lambda i: ctx.fhe_mult_scalar(xs[i], 123456789, out=outs[i]), "fhe_mult_scalar"),
        ("multconstvec_pairwise_into", lambda i: ctx.fhe_mult_plain(xs[i], pts[i], 1, out=outs[i], stream=stream), "fhe_mult_plain, one plaintext per ciphertext"),
    )
    reps = max(8, args.steps)
    for name, fn, what in ops:
        for i in range(max(args.warmup, 3)):
            fn(i % NSET)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for i in range(reps):
            fn(i % NSET)
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / reps
        t4, line = PAPER_TABLE1_T4_S[name]
        print(json.dumps({"table1": True, "operation": name, "call": what, "metric": "CipherTensor latency", "value": ms / 1e3,
                          "unit": "s", "higher_is_better": False, "us_per_ciphertext": ms * 1e3 / B,
                          "config": {"workload": "paper Table 1 shape: cnum=4, N=65536, logQ=1024, logP=1024, logp=60 (PAPER.md:711-721)"},
                          "paper_t4_s": t4, "paper_cite": f"PAPER.md:{line}", "paper_hardware": "Tesla T4, Numba (context, not a target)",
                          "dtype": "u32 (exact integer)", "data": "synthetic", "reps": reps}), flush=True)
    return 0

# ---- all five BASELINE.json configs, one JSON line each (context for the parity cases; the metric is quoted on C5) --------
def run_configs(args):
    import numpy as np
    import torch
    import synth
    import paper_2607_05920_b200 as fhe

    rank, local_rank, world = dist_env()
    if rank != 0:
        return 0
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    stream = torch.cuda.current_stream(dev)
    cfgs = (   # name, N, logQ, logP, t, batch, call
        ("c1", 1 << 10, 128, 128, 0, 1, "mult_relin_rescale"),
        ("c2", 1 << 13, 218, 32, 0, 64, "polymul"),
        ("c3", 1 << 15, 620, 620, 0, 8, "mult_relin_rescale"),
        ("c4", 1 << 14, 437, 437, 65537, 16, "mult_relin"),
        ("c5", 1 << 16, 1240, 1240, 0, 4, "mult_relin_rescale"),
    )
    for name, N, logQ, logP, t, B, call in cfgs:
        ctx = fhe.Context(N, logQ, logP, t)
        g = synth.rng(77)

        def limbs(lead, bits):
            return torch.from_numpy(synth.uniform_limbs(g, lead, N, bits).view(np.int32)).to(dev)   # < 2^bits <= the modulus

        if call == "polymul":
            a, b = limbs((B,), logQ), limbs((B,), logQ)
            out = torch.empty_like(a)
            fn = lambda: ctx.fhe_polymul(a, b, out=out, stream=stream)
            unit = "polymuls/s"
        else:
            a, b = limbs((B, 2), logQ), limbs((B, 2), logQ)
            ctx.fhe_set_evk(limbs((2,), logQ + logP))
            out = torch.empty_like(a)
            fn = lambda: ctx.fhe_mult_relin_rescale(a, b, 40 if t == 0 else 0, out=out, stream=stream)
            unit = "ops/s"
        for _ in range(max(args.warmup, 3)):
            fn()
        torch.cuda.synchronize()
        l0 = ctx.launch_count()
        reps = max(args.steps, 10)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / reps
        print(json.dumps({"configs": True, "config": {"workload": name, "N": N, "logQ": logQ, "logP": logP, "t": t, "batch": B, "call": call},
                          "metric": unit, "value": B / (ms / 1e3), "unit": unit, "ms_per_step": ms, "us_per_item": ms * 1e3 / B,
                          "launches_per_step": (ctx.launch_count() - l0) // reps, "L": ctx.L, "K": ctx.K_pm if call == "polymul" else [ctx.K1, ctx.K2],
                          "dtype": "u32 (exact integer)", "data": "synthetic"}), flush=True)
        del ctx, a, b, out
        torch.cuda.empty_cache()
    return 0


# ---- profiles/: turn an exported ncu capture of this command into the committed summaries --------------------------------
KERNEL_CLASS_PATTERNS = (   # substring of the kernel name -> bench.py's kernel class
    ("DecEpi", "decompose"), ("decompose_small", "decompose"), ("CrtEpi", "crt"), ("crt_exact", "crt"), ("crt_small", "crt"),
    ("ntt_row_fused", "pointwise"), ("ntt_whole", "pointwise"), ("rescale_kernel", "rescale"),
)


def kernel_class(name: str):
    for pat, cls in KERNEL_CLASS_PATTERNS:
        if pat in name:
            return cls
    if "ntt_col" in name or "ntt_row_fwd" in name or "ntt_row_inv" in name:
        # ntt_col2_kernel<LN, INV, PM> / ntt_col_kernel<LN, INV>: the second template argument is the direction
        import re
        m = re.search(r"<\s*\d+\s*,\s*(\w+)\s*[,>]", name)
        inv = "ntt_row_inv" in name or (m is not None and m.group(1) in ("1", "true"))
        return "ntt_inv" if inv else "ntt_fwd"
    return None


def summarise_ncu(raw_csv: str, capture_name: str):
    """raw_csv = `ncu -i <capture>.ncu-rep --page raw --csv` of `ncu --set full ... python bench.py ...` (one step's launches).
    Writes profiles/dram_traffic.csv (read back by the roofline line) and prints a markdown table for profiles/*.md."""
    import csv
    with open(raw_csv) as f:
        rows = list(csv.reader(f))
    hdr, body = rows[0], rows[2:]
    col = {h: i for i, h in enumerate(hdr)}
    def num(r, key):
        v = r[col[key]].replace(",", "") if key in col else ""
        try:
            return float(v)
        except ValueError:
            return 0.0
    unit = {h: rows[1][i] for h, i in col.items()}
    def to_bytes(v, u):
        return v * {"byte": 1, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(u, 1)
    per = {}
    lines = ["| # | kernel | class | us | DRAM read MB | DRAM write MB | dram % of peak | issue active % | tensor pipe % | regs |", "|---|---|---|---|---|---|---|---|---|---|"]
    for n, r in enumerate(body):
        name = r[col["Kernel Name"]]
        cls = kernel_class(name)
        rd = to_bytes(num(r, "dram__bytes_read.sum"), unit.get("dram__bytes_read.sum", "byte"))
        wr = to_bytes(num(r, "dram__bytes_write.sum"), unit.get("dram__bytes_write.sum", "byte"))
        us = num(r, "gpu__time_duration.sum") * {"ns": 1e-3, "us": 1.0, "ms": 1e3}.get(unit.get("gpu__time_duration.sum", "us"), 1.0)
        dram_pct = num(r, "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed")
        lines.append(f"| {n} | `{name[:60]}` | {cls} | {us:.1f} | {rd / 1e6:.1f} | {wr / 1e6:.1f} | {dram_pct:.1f} | "
                     f"{num(r, 'smsp__issue_active.avg.pct_of_peak_sustained_active'):.1f} | "
                     f"{num(r, 'sm__pipe_tensor_cycles_active.avg.pct_of_peak_sustained_active'):.1f} | {int(num(r, 'launch__registers_per_thread'))} |")
        if cls:
            d = per.setdefault(cls, [0, 0.0, 0.0])
            d[0] += 1; d[1] += rd + wr; d[2] += us
    head = kernel_source_hash()
    with open(TRAFFIC_CSV, "w") as f:
        f.write("# DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) per launch and kernel class, one C5 step; written by\n"
                "# `python bench.py --ncu-raw <csv> --capture-name <name>` from an `ncu --set full` capture of bench.py itself\n")
        f.write("class,launches_per_step,dram_bytes_per_launch,kernel_source_sha256_16,capture\n")
        for cls, (cnt, byts, us) in sorted(per.items()):
            f.write(f"{cls},{cnt},{byts / cnt:.0f},{head},{capture_name}\n")
    print("\n".join(lines))
    print()
    print("| class | launches | DRAM MB per step | us per step (serialised, cold cache) | share |")
    print("|---|---|---|---|---|")
    tot = sum(v[2] for v in per.values())
    for cls, (cnt, byts, us) in sorted(per.items()):
        print(f"| {cls} | {cnt} | {byts / 1e6:.1f} | {us:.1f} | {us / tot:.3f} |")
    print(f"| total | {sum(v[0] for v in per.values())} | {sum(v[1] for v in per.values()) / 1e6:.1f} | {tot:.1f} | 1 |")
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c5", choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true",
                    help="standalone polymul sweep N = 2^12..2^16 x logQ in {64, 256, 620, 1240, 2480}: one JSON line per cell")
    ap.add_argument("--table1", action="store_true",
                    help="the operations of the paper's Table 1 at the paper's shape (cnum = 4, N = 2^16, logQ = 1024): one JSON line each")
    ap.add_argument("--configs", action="store_true", help="time the call of each of the five BASELINE.json configs: one JSON line each")
    ap.add_argument("--ncu-raw", default=None, help="exported raw page (csv) of an ncu --set full capture of this command: "
                                                    "write profiles/dram_traffic.csv and print the summary tables")
    ap.add_argument("--capture-name", default="capture")
    args = ap.parse_args()
    if args.ncu_raw:
        return summarise_ncu(args.ncu_raw, args.capture_name)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours" and not args.sweep and not args.table1 and not args.configs:
        # plain `python bench.py --gpus N`: become the N-rank launch the contract describes (one process per GPU)
        port = os.environ.get("MASTER_PORT", "29511")
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", port, os.path.abspath(__file__)] + sys.argv[1:]
        os.execv(sys.executable, cmd)
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    if args.table1:
        return run_table1(args)
    if args.configs:
        return run_configs(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
