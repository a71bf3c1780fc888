"""bench.py -- one J+K build per step through the C ABI (include/pbc_jk.h), timed on a B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload water64] [--impl reference]

A "step" is one pass of the whole hot path (density prep, real-space J-engine
and K quartet kernels of every class, reciprocal-space rho(G)/J/K, SELF term, finalise) for one
density matrix on a fixed geometry.  pbc_jk_create (A1-A3, the paper's "initialization") is timed
separately.  Rank 0 prints ONE JSON line:

  metric   primitive quartet-images evaluated in real space (J + K) per second of J+K build
           (BASELINE.json: "J+K build seconds per SCF iteration & quartets/s"); ms_per_step is the
           J+K build time itself.
  value    device-resident leg: P, J, K live in HBM; CUDA events on the build's stream.
  e2e      same through pbc_jk_build_host with pinned HOST buffers (P up, J and K down, per step).
  roofline the kernel family with the largest share of the step -- the reciprocal-space K GEMMs (FP64 tensor
           cores, DMMA) or the real-space quartet kernels (FP64 FMA pipe) -- with both families printed
           (DESIGN.md section 7); peaks measured live by the helper library libpbc_jk_benchpeaks.so.
  cpu_baseline  the fp64 oracle, as it stands, on a bounded sample of output shell blocks, and the
           extrapolation of that sample to a full build.

--impl reference times the oracle alone (the reference arm of this tier).
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

METRIC = "jk_build_primitive_quartets_per_s"
UNIT = "quartets/s"


# ----------------------------------------------------------------------------------------------
# algorithmic flop model per primitive quartet-image
# ----------------------------------------------------------------------------------------------
def ncart(l):
    return (l + 1) * (l + 2) // 2


def nherm(L):
    return (L + 1) * (L + 2) * (L + 3) // 6


def _cart(l):
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]


def _eterms(la, lb):
    """number of non-zero separable E^{ab}_t over all component pairs (= n_ab * zbar_ab)"""
    return sum((a[0] + b[0] + 1) * (a[1] + b[1] + 1) * (a[2] + b[2] + 1) for a in _cart(la) for b in _cart(lb))


def flops_base(L):
    """merged Boys values (two arguments) + Hermite R recursion (eq 47-51) for total order L"""
    boys = 60 + 6 * L
    rec = 0
    for m in range(L):                      # level m builds orders 1..L-m from level m+1
        for n in range(1, L - m + 1):
            for t in range(n, -1, -1):
                for u in range(n - t, -1, -1):
                    v = n - t - u
                    k = t if t > 0 else (u if u > 0 else v)
                    rec += 1 + (2 if k > 1 else 0)      # one MUL, one FMA when the index exceeds 1
    return boys + rec


def flops_j(LB, LK):
    return flops_base(LB + LK) + 2 * nherm(LB) * nherm(LK)


def flops_k(la, lb, lc, ld):
    nab, ncd = ncart(la) * ncart(lb), ncart(lc) * ncart(ld)
    fma = nherm(la + lb) * _eterms(ld, lc) + ncd * _eterms(la, lb) + nab * ncd
    return flops_base(la + lb + lc + ld) + 2 * fma


def class_flops(cs):
    return flops_j(*cs["l"]) if cs["kind"] == "J" else flops_k(*cs["l"])


# ----------------------------------------------------------------------------------------------
# helpers
# ----------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.rows = []
        self.stop = threading.Event()
        self.th = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                f = [x.strip() for x in out.strip().split(",")]
                if len(f) >= 7:
                    self.rows.append(f)
            except Exception:
                pass
            self.stop.wait(0.2)

    def __enter__(self):
        self.th.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.th.join(timeout=6)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm = sorted(float(r[0]) for r in self.rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[3 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]),
                "power_w_max": max(float(r[2]) for r in self.rows), "reasons": reasons, "samples": len(self.rows)}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


def _ncu_traffic(kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed raw-page CSV extract of an
    `ncu --set full` capture (profiles/r2_ncu_dram_bytes.csv: kernel, launches, bytes_read, bytes_write; written by the
    command named in profiles/r2_ncu_dram_bytes.md).  None (= not measured) when the file or the kernel is absent."""
    p = os.path.join(ROOT, "profiles", "r2_ncu_dram_bytes.csv")
    if not os.path.exists(p):
        return None
    import csv
    for row in csv.DictReader(open(p)):
        if row["kernel"] == kernel:
            return (float(row["bytes_read"]) + float(row["bytes_write"])) / max(1.0, float(row["launches"]))
    return None


def _pair_traffic():
    """DRAM bytes of one dgemm_kernel<0,0> + dgemm_kernel<0,1> launch pair (the unit of the GEMM roofline), or None"""
    a, b = _ncu_traffic("dgemm_kernel<0,0>"), _ncu_traffic("dgemm_kernel<0,1>")
    return a + b if a is not None and b is not None else None


def h_nb(st, n):
    """G vectors per reciprocal-space batch as pbc_jk_create sizes them (stacks <= 12 GB, at most 64)"""
    np_ = ((n + 63) // 64) * 64
    nb = max(1, min(64, int(12.0e9 // (np_ * np_ * 16)), max(st["n_g"], 1)))
    return (nb // 16) * 16 if nb >= 16 else nb


def _oracle_sample_blocks(wl, nblk, seed=12345):
    """Seeded sample of output shell blocks covering every (l_mu, l_nu) class of the workload."""
    rng = np.random.default_rng(seed)
    by_l = {}
    for s, l in enumerate(wl.sh_l):
        by_l.setdefault(int(l), []).append(s)
    classes = [(a, b) for a in sorted(by_l) for b in sorted(by_l) if a >= b]
    blocks = []
    k = 0
    while len(blocks) < nblk:
        la, lb = classes[k % len(classes)]
        blocks.append((int(rng.choice(by_l[la])), int(rng.choice(by_l[lb]))))
        k += 1
    return blocks


def _time_oracle(wl, P, target_s=15.0, max_blocks=256):
    """The oracle as it stands on a bounded sample: its real-space (SR) part -- the part the metric's
    quartets belong to -- for a growing number of sampled output shell blocks until ~target_s of wall
    time was spent.  (The oracle's reciprocal-space pass costs the same for one block as for all of
    them -- it rebuilds rho_mn(G) of every pair for every G -- so it is left out of the sample.)
    Returns (quartets, seconds, nblocks, cores)."""
    import oracle
    oracle.build()
    cores = oracle.num_threads()
    nblk, q, dt = 1, 0, 0.0
    while True:
        blocks = _oracle_sample_blocks(wl, nblk)
        t0 = time.perf_counter()
        r = oracle.jk(wl, P, blocks=blocks, parts="sr")
        dt = time.perf_counter() - t0
        q = r["counts"]["quartets_J"] + r["counts"]["quartets_K"]
        if dt >= 0.5 * target_s or nblk >= max_blocks:
            break
        nblk = min(max_blocks, max(nblk + 1, int(nblk * min(8.0, 0.8 * target_s / max(dt, 1e-3)))))
    return q, dt, nblk, cores


def _extrapolate_oracle(wl, P, nblk, n_g_half):
    """the sampled oracle times extrapolated to a full build, labelled as such.  Real space: the sample is
    stratified by output class (l_mu >= l_nu), so each class is timed on its own sampled blocks and scaled by the number
    of ordered output blocks of that class.  Reciprocal space: the oracle's G pass costs the same for one block as for
    all (it rebuilds rho_mn(G) of every pair per G), so a short window of G is timed and scaled by the G count."""
    import oracle
    blocks = _oracle_sample_blocks(wl, nblk)
    ls = [int(l) for l in wl.sh_l]
    cnt_l = {l: ls.count(l) for l in set(ls)}
    per_class = {}
    for (a, b) in blocks:
        per_class.setdefault((ls[a], ls[b]), []).append((a, b))
    sr_full = 0.0
    for (la, lb), blk in per_class.items():
        t0 = time.perf_counter()
        oracle.jk(wl, P, blocks=blk, parts="sr")
        dt = time.perf_counter() - t0
        n_ordered = cnt_l[la] * cnt_l[lb] * (1 if la == lb else 2)
        sr_full += dt / len(blk) * n_ordered
    # G window: |G| up to about 2.4 reciprocal-lattice spacings (a few dozen vectors)
    g_win = 2.4 * 2.0 * np.pi / float(np.linalg.norm(wl.cell, axis=1).max())
    t0 = time.perf_counter()
    r = oracle.jk(wl, P, blocks=blocks[:1], parts="lr", g_cut=g_win)
    dt = time.perf_counter() - t0
    ng = max(1, r["counts"]["n_G"])
    lr_full = dt / ng * (2 * n_g_half)
    return {"extrapolated_full_build_seconds": sr_full + lr_full,
            "extrapolation": f"EXTRAPOLATED: real space {sr_full:.0f} s (per-class sampled seconds x ordered blocks of the class), "
                             f"reciprocal space {lr_full:.0f} s ({dt / ng:.3f} s per G over {ng} G x {2 * n_g_half} G of the full sphere)"}


def _workload_and_density(name):
    from paper_2410_22278_b200 import workloads
    wl = workloads.get(name)
    return wl


def run_reference(args, rank):
    """--impl reference: the oracle alone, each step a bounded sample of the workload."""
    if rank != 0:
        return
    import oracle
    from paper_2410_22278_b200 import workloads
    oracle.build()
    wl = workloads.get(args.workload)
    S = oracle.overlap(wl)
    P = workloads.density_from_orbitals(wl.orbitals_seed(), S)
    # size the sample once (about 10 s), then W + K steps on exactly that sample
    _, dt0, nblk, cores = _time_oracle(wl, P, target_s=10.0)
    blocks = _oracle_sample_blocks(wl, nblk)
    times, quartets = [], 0
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        r = oracle.jk(wl, P, blocks=blocks, parts="sr")
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt)
            quartets = r["counts"]["quartets_J"] + r["counts"]["quartets_K"]
    sec = sum(times) / len(times)
    val = quartets / sec
    sample = f"real-space part of {nblk} seeded output shell blocks of {args.workload} (J and K), fp64"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "nbf": wl.nbf, "natom": wl.natom, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="water64",
                    help="tiny | water8 | si64 | water64 (config 4, the 192-atom metric config) | water343")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--precision", default="fp64", choices=["fp64", "mixed"],
                    help="mixed: real-space K quartets below the switch in fp32 (PAPER 3.5 L817-821)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    from paper_2410_22278_b200 import workloads
    from paper_2410_22278_b200.binding import PbcJK, allreduce_jk, bench_peaks, load

    load()                                             # fails loudly if libpbc_jk.so is missing
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    wl = workloads.get(args.workload)
    h = PbcJK(wl, precision=1 if args.precision == "mixed" else 0)
    n = h.nbf
    S = h.overlap()                                    # the library's own crystalline overlap (A3)
    P = workloads.density_from_orbitals(wl.orbitals_seed(), S)
    # N > 1: ONE build sharded over the ranks (real-space blocks / bras and G batches dealt round-robin),
    # partial matrices summed by one all-reduce of [J; K] -- total work fixed: strong scaling
    if world > 1:
        h.set_shard(rank, world)

    Pd = torch.from_numpy(P).cuda()
    JK = torch.empty((2, n, n), dtype=torch.float64, device="cuda")      # J and K back to back: one all-reduce message
    Jd, Kd = JK[0], JK[1]
    Ph = torch.from_numpy(P).pin_memory()
    Jh = torch.empty((n, n), dtype=torch.float64).pin_memory()
    Kh = torch.empty((n, n), dtype=torch.float64).pin_memory()
    flush = torch.empty(512 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")   # 512 MB > 126 MB L2
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        h.build(Pd, Jd, Kd)
        if world > 1:
            allreduce_jk(Jd, Kd)

    h.set_profile(True)                                # an event pair per class launch and per GEMM pair: the roofline times
    # ---------------- device-resident leg ----------------
    for _ in range(args.warmup):
        flush.zero_()
        step()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    cls_ms = {}
    gemm_ms = 0.0
    with ClockSampler(local_rank) as clocks:
        barrier()
        for i in range(args.steps):
            flush.zero_()                              # L2 flush between timed iterations (outside the events)
            ev[i][0].record(stream)
            step()
            ev[i][1].record(stream)
            # per-launch times of this step (events live in the handle; read before the next build)
            ev[i][1].synchronize()
            for cs in h.class_stats():
                key = (cs["kind"], cs["l"])
                e = cls_ms.setdefault(key, dict(cs, ms=0.0))
                e["ms"] += cs["ms"] / args.steps
            gemm_ms += h.stats()["ms_lr_gemm"] / args.steps
        barrier()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    st = h.stats()
    t = torch.tensor([sum(step_ms)], dtype=torch.float64, device="cuda")
    q = torch.tensor([st["quartets_j"] + st["quartets_k"]], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(q, op=dist.ReduceOp.SUM)       # every quartet is evaluated by exactly one rank
    total_ms = float(t.item())
    ms_per_step = total_ms / args.steps
    quartets = float(q.item())
    value = quartets / (ms_per_step * 1e-3)

    # ---------------- end-to-end leg: host buffers through pbc_jk_build_host ----------------
    h.set_profile(False)

    def step_host():
        h.build_host_ptr(Ph.data_ptr(), Jh.data_ptr(), Kh.data_ptr())     # synchronous: P up, J and K down
        if world > 1:                                  # NCCL reduces device memory: partial J, K up again, sums back down
            Jd.copy_(Jh, non_blocking=True); Kd.copy_(Kh, non_blocking=True)
            allreduce_jk(Jd, Kd)
            Jh.copy_(Jd, non_blocking=True); Kh.copy_(Kd, non_blocking=True)
            torch.cuda.synchronize()

    for _ in range(2):
        step_host()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        flush.zero_()
        step_host()
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / args.steps
    t = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    e2e_s = float(t.item())
    if world == 1:
        dJ = float((Jh.cuda() - Jd).abs().max().item())
        dK = float((Kh.cuda() - Kd).abs().max().item())
        assert dJ == 0.0 and dK == 0.0, "host-buffer and device-buffer builds differ"

    if rank == 0:
        peaks, peaks_kind = _peaks()
        # ---------------- roofline: both kernel families, the one with the larger share of the step on top ----------------
        pk = bench_peaks(20000)                        # DFMA / FFMA / DMMA micro-benchmarks on this device, TFLOP/s
        sm_max = float(peaks.get("sm_max_mhz", 1965.0))
        fp64_nominal = 148 * 64 * 2 * sm_max * 1e6 * 1e-12      # 148 SMs x 64 FP64 FMA lanes x 2 flop x clock
        fp32_nominal = 2.0 * fp64_nominal
        # FP64 tensor (DMMA) peak derived as the contract asks: measured bf16 peak x nominal ratio 45 / 2250 TFLOP/s
        dmma_derived = float(peaks.get("bf16_tflops", 1590.0)) * 45.0 / 2250.0
        rows = sorted(cls_ms.values(), key=lambda c: -c["ms"])
        sr_ms = sum(c["ms"] for c in rows)
        sr_flop = sum(class_flops(c) * c["quartets"] for c in rows)
        fam = {}
        for c in rows:
            f = fam.setdefault(c["kind"], {"ms": 0.0, "flop": 0.0, "quartets": 0})
            f["ms"] += c["ms"]; f["flop"] += class_flops(c) * c["quartets"]; f["quartets"] += c["quartets"]
        sr_tf = sr_flop / (sr_ms * 1e-3) * 1e-12 if sr_ms > 0 else 0.0
        # reciprocal-space K (A8): per G slot  Y = L^T A' (2 r N^2 flop)  and  K += Y^T Y on the lower triangle (r N (N+1));
        # slots = Re and Im of every G of this rank's batches, plus the SELF slot; r = rank of the factor of P'
        r_p = int(st["rank_p"])
        slots = 2 * ((st["n_g"] + world - 1) // world if world > 1 else st["n_g"]) + (1 if rank == 0 else 0)
        gemm_flop = (2.0 * r_p * n * n + r_p * n * (n + 1.0)) * slots
        gemm_tf = gemm_flop / (gemm_ms * 1e-3) * 1e-12 if gemm_ms > 0 else 0.0
        n_gemm_launch = 2 * ((st["n_g"] + h_nb(st, n) - 1) // h_nb(st, n) + 1)
        real_space = {"bound": "alu", "kernel": "sr_k_kernel<*> + sr_j_kernel<*> (one launch per class)", "ms": sr_ms,
                      "achieved": sr_tf, "peak": fp64_nominal, "unit": "TFLOP/s", "frac": sr_tf / fp64_nominal,
                      "share_of_step": sr_ms / ms_per_step,
                      "peak_kind": f"FP64 FMA nominal: 148 SM x 64 lanes x 2 x {sm_max:.0f} MHz; DFMA micro-benchmark on this box "
                                   f"{pk['fp64_fma']:.2f} TFLOP/s (FFMA {pk['fp32_fma']:.2f})",
                      "families": {k: {"ms": v["ms"], "quartets": v["quartets"],
                                       "tflops": v["flop"] / (v["ms"] * 1e-3) * 1e-12 if v["ms"] > 0 else 0.0} for k, v in fam.items()},
                      "top_classes": [{"kind": c["kind"], "l": list(c["l"]), "ms": round(c["ms"], 3), "quartets": c["quartets"],
                                       "tflops": round(class_flops(c) * c["quartets"] / (c["ms"] * 1e-3) * 1e-12, 3) if c["ms"] > 0 else 0.0}
                                      for c in rows[:8]]}
        if args.precision == "mixed":
            real_space["fp32_quartets_k"] = st["quartets_k_fp32"]
            real_space["fp32_share_of_k_quartets"] = st["quartets_k_fp32"] / max(1, st["quartets_k"])
            real_space["fp32_peak"] = fp32_nominal
        lr_gemm = {"bound": "tensor", "kernel": "dgemm_kernel<0,0> + dgemm_kernel<0,1> (mma.sync.m8n8k4.f64, one pair per G batch)",
                   "ms": gemm_ms, "achieved": gemm_tf, "peak": pk["fp64_dmma"], "unit": "TFLOP/s",
                   "frac": gemm_tf / pk["fp64_dmma"] if pk["fp64_dmma"] > 0 else 0.0, "share_of_step": gemm_ms / ms_per_step,
                   "peak_kind": f"FP64 tensor (DMMA) micro-benchmark on this box; derived from MEASURED_PEAKS bf16 x 45/2250: "
                                f"{dmma_derived:.1f} TFLOP/s ({peaks_kind})",
                   # context for the fraction: DMMA and DFMA warps side by side (sum of both rates: one shared
                   # FP64 pipe if it equals the peak) and the kernel's inner loop without its global loads
                   "fp64_probes_tflops": {"dmma": round(pk["fp64_dmma"], 2), "dfma": round(pk["fp64_fma"], 2),
                                          "dmma_and_dfma_side_by_side": round(pk["fp64_mixed_pipe"], 2),
                                          "gemm_inner_loop_no_global_loads": round(pk["fp64_dmma_loop"], 2)},
                   "flop_per_launch_pair": gemm_flop / max(1, n_gemm_launch // 2), "rank_of_P": r_p, "g_slots": slots,
                   "ms_per_launch_pair": gemm_ms / max(1, n_gemm_launch // 2),
                   "traffic": _pair_traffic() if args.workload == "water64" and world == 1 else None,   # the capture is water64's
                   "ms_lr_phase": st["ms_lr"]}
        top, other = (lr_gemm, real_space) if gemm_ms >= sr_ms else (real_space, lr_gemm)
        roofline = dict(top)
        roofline.setdefault("traffic", None)               # not measured for the real-space family (compute-bound: DESIGN.md 7)
        roofline["other_family"] = other
        # ---------------- CPU baseline: the oracle on a bounded sample ----------------
        cpu = None
        if not args.no_cpu_baseline:
            q, dt, nblk, cores = _time_oracle(wl, P, target_s=15.0)
            cpu = {"value": q / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                   "sample": f"real-space part of {nblk} seeded output shell blocks of {args.workload}: {q} primitive quartet-images in {dt:.1f} s "
                             f"(the oracle screens at 1e-18, so it evaluates more quartets per block than the GPU path)"}
            cpu.update(_extrapolate_oracle(wl, P, nblk, st["n_g"]))
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak" if world == 1 else "strong",
            "vs_baseline": None,
            "dtype": "f64" if args.precision == "fp64" else "f64+f32", "data": "synthetic",
            "config": {"workload": args.workload, "natom": wl.natom, "nshell": wl.nshell, "nbf": n, "omega": wl.omega,
                       "n_g_half": st["n_g"], "prim_pair_images": st["n_prim_pairs"], "precision": args.precision,
                       "l2": "512 MB flush write between timed iterations", "parallelism": "1 gpu" if world == 1 else f"one build sharded over {world} GPUs (K blocks, J bras, G batches round-robin) + "
                                                                           "one all-reduce of [J; K]"},
            "jk_build_seconds": ms_per_step * 1e-3, "create_seconds": st["create_seconds"],
            "quartets_per_step": {"J": st["quartets_j"], "K": st["quartets_k"],
                                  "candidates_J": st["candidates_j"], "candidates_K": st["candidates_k"]},
            "phase_ms": {k: st[k] for k in ("ms_density", "ms_sr_j", "ms_sr_k", "ms_lr", "ms_total")},
            "step_ms": [round(x, 3) for x in step_ms],
            "e2e": {"value": quartets / e2e_s, "unit": UNIT, "ms_per_step": e2e_s * 1e3,
                    "h2d_bytes_per_step": n * n * 8, "d2h_bytes_per_step": 2 * n * n * 8},
            "gpu_launches": int(st["n_launches"]) * args.steps,
            "clocks": clocks.summary(), "peaks": peaks_kind,
            "roofline": roofline, "cpu_baseline": cpu,
        }
        print(json.dumps(line), flush=True)
    h.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
