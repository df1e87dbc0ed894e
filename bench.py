#!/usr/bin/env python
"""bench.py -- throughput of the Hermitian PSD-cone projection (the hot path of arxiv/paper_2606_20519).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

One "step" = one pass of the whole hot path (S0..S10) over one cone list of
BASELINE.json's configs (default: config 3, the single n=625 block the metric is quoted on).
Prints ONE JSON line (see the task contract): `value` = projections/s with inputs resident in HBM,
`e2e` = the same through hpsd_project_host with host buffers, `roofline` for the dominant kernel
(live CUDA-event stage timers inside the library), `cpu_baseline` = the oracle on the host cores.
`--impl reference` times the CPU oracle alone.  Multi-GPU: a single block does not shard
(DESIGN.md §Multi-GPU): N ranks run N independent replicas ("weak").
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402  (seeded input generators only; none of the method's arithmetic)

METRIC = "hermitian_psd_projections_per_sec"
UNIT = "projections/s"
L2_FLUSH_BYTES = 512 << 20


def f_alg(n: int, kpos: int) -> float:
    """Algorithmic real flops of one projection: reduction + tridiagonal D&C +
    one back-transform of the kpos kept columns + HERK.  Extra work of a variant is not counted."""
    if n <= 1:
        return 0.0
    return (16.0 / 3.0) * n ** 3 + (4.0 / 3.0) * n ** 3 + 8.0 * n * n * kpos + 4.0 * n * n * kpos


# stage -> the part of f_alg that stage carries (flops), used for the dominant-kernel roofline.
# route(n) -> "jacobi" | "medium" | "cluster" | "panel" | "two_stage"
def stage_flops(stage: str, sizes, kpos, route) -> float:
    tot = 0.0
    for n, k in zip(sizes, kpos):
        r = route(n)
        large = r in ("cluster", "panel", "two_stage")
        if stage == "S2S3_tridiag_panel" and large:
            if r == "cluster":
                tot += (16.0 / 3.0) * n ** 3     # the cluster-resident kernel does both halves of the reduction
            elif r == "panel":
                tot += (8.0 / 3.0) * n ** 3      # the mat-vec half
            else:
                tot += 4.0 * n * n * 32          # panel QR of the two-stage reduction: sum_k 8 m b^2
        elif stage == "S2_her2k_trailing" and large:
            tot += ((16.0 if r == "two_stage" else 8.0) / 3.0) * n ** 3      # two-stage: HEMM + HER2K
        elif stage == "S4_stedc" and large:
            tot += (4.0 / 3.0) * n ** 3
        elif stage == "S5S6_backtransform" and large:
            tot += 8.0 * n * n * k
        elif stage == "S7S8_herk_pack" and large:
            tot += 4.0 * n * n * k
        elif stage in ("S9_jacobi", "S10_householder_ql") and r in ("jacobi", "medium"):
            tot += f_alg(n, k)
        # S3_bulge_chasing and S5_backtransform_q2 are extra work of the two-stage variant: no share of f_alg
    return tot


# extra real flops a variant spends beyond f_alg (reported, never credited): bulge chasing 24 b n^2, second back-transform 8 n^2 k
def variant_flops(stage: str, sizes, kpos, route) -> float:
    tot = 0.0
    for n, k in zip(sizes, kpos):
        if route(n) != "two_stage":
            continue
        if stage == "S3_bulge_chasing":
            tot += 24.0 * 32 * n * n
        elif stage == "S5_backtransform_q2":
            tot += 8.0 * n * n * k
    return tot


def panel_bytes(n: int) -> float:
    """Algorithmic bytes of the panel kernel for one n x n block: per column c the Hermitian mat-vec reads the
    stored lower triangle (diagonal included) of the (n-c-1) x (n-c-1) trailing matrix once, 16 B per entry."""
    return float(sum(16 * (m * (m + 1) // 2) for m in range(1, n)))


def measured_hbm_gbs():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (driver-measured copy bandwidth, burst)"
    except (OSError, KeyError, ValueError):
        return 6650.0, "fallback 6.65 TB/s of B200_PROFILING.md (MEASURED_PEAKS.json absent)"


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed ncu --set full
# captures of THIS round's kernels (profiles/r2_ncu_full.md lists kernel, workload, command and both counters);
# None where no capture exists for that kernel and workload
NCU_TRAFFIC = {
    ("tridiag_cluster_kernel", 3): {"bytes_per_launch": 3.18e6, "source": "profiles/r2_ncu_full.md (n=625, whole reduction in one launch)"},
    ("tridiag_panel_kernel", 5): {"bytes_per_launch": 2.019e9, "source": "profiles/r2_ncu_full.md (first panel of n=4096: 1913 MB read + 106 MB written; algorithmic 2.1 GB)"},
}


def ncu_traffic(kernel: str, cfg: int):
    e = NCU_TRAFFIC.get((kernel, cfg)) or {}
    return e.get("bytes_per_launch"), e.get("source")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "20", "-i", str(self.index)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        for r in self.rows:
            if len(r) < 8:
                continue
            try:
                sm.append(float(r[1])); mx.append(float(r[2])); pw.append(float(r[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(cfg: int):
    """A bounded sample of the workload for the CPU oracle (about 10-30 s): (sizes, matrices, scale,
    description); time(full workload) ~ scale * time(sample) by the n^3 cost law."""
    w = workloads.make(cfg) if cfg in (1, 2, 3) else None
    if cfg == 1:
        return w.sizes, [b.X for b in w.blocks], 1.0, "the whole workload (one n=16 block), repeated"
    if cfg == 2:
        return w.sizes[:64], [b.X for b in w.blocks[:64]], 4.0, "64 of the 256 n=81 blocks; time x4"
    if cfg == 3:
        return w.sizes, [b.X for b in w.blocks], 1.0, "the whole workload (one n=625 block)"
    if cfg == 4:
        rng = np.random.default_rng(workloads.BASE_SEED + 4)
        b = workloads.gue_like(rng, 1296, 1.0 / 36.0)
        scale = (1296.0 ** 3 + 2401.0 ** 3 + 64 * 36.0 ** 3) / 1296.0 ** 3
        return [1296], [b.X], scale, f"the n=1296 block only; time x{scale:.3f} (sum n^3 / 1296^3)"
    rng = np.random.default_rng(workloads.BASE_SEED + 5)
    b = workloads.from_spectrum(rng, workloads.spectrum_clustered(rng, 1024, n_big=16, n_clusters=8, mult=32))
    return [1024], [b.X], 64.0, "a config-5-type block (clusters of 32 repeats) at n=1024; time x64 ((4096/1024)^3)"


def run_oracle(cfg: int, steps: int, warmup: int, min_seconds: float = 0.0):
    """Times the oracle as it stands on the host cores.  Returns (projections/s, s per step, cores, sample)."""
    import oracle
    oracle.build()
    sizes, mats, scale, desc = oracle_sample(cfg)
    sv = np.concatenate([oracle.pack(m) for m in mats])
    threads = oracle.max_threads()
    for _ in range(warmup):
        oracle.project(sizes, sv, nthreads=threads)
    times = []
    t_all = time.perf_counter()
    while len(times) < steps or (time.perf_counter() - t_all) < min_seconds:
        t0 = time.perf_counter()
        oracle.project(sizes, sv, nthreads=threads)
        times.append(time.perf_counter() - t0)
        if len(times) >= max(steps, 1) and min_seconds <= 0.0:
            break
    per_step = scale * sum(times) / len(times)
    return 1.0 / per_step, per_step, threads, f"{desc}; {len(times)} timed run(s), {threads} OpenMP thread(s)"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-secondary", action="store_true", help="skip the n=4096 ms/projection figure")
    ap.add_argument("--only-n4096", action="store_true", help="secondary figure: config 5 only (skip configs 1, 2, 4)")
    ap.add_argument("--no-routes", action="store_true", help="skip the one-stage vs two-stage table")
    ap.add_argument("--two-stage", type=int, default=0, choices=[0, 1, 2], help="library option two_stage for the timed workload")
    ap.add_argument("--two-stage-min-n", type=int, default=1024)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = args.config
    wname = {1: "cfg1: 1 x n=16 Haar/Gaussian spectrum", 2: "cfg2: 256 x n=81 GUE-like",
             3: "cfg3: 1 x n=625 ADMM-like low-rank spectrum", 4: "cfg4: n=1296 + n=2401 + 64 x n=36 GUE-like",
             5: "cfg5: 1 x n=4096 clustered spectrum"}[cfg]

    # ------------------------------------------------------------------ reference arm = the oracle
    if args.impl == "reference":
        if rank != 0:
            return
        value, per_step, threads, sample = run_oracle(cfg, max(args.steps, 1), min(args.warmup, 1))
        print(json.dumps({
            "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": per_step * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wname, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0,
        }))
        return

    # ------------------------------------------------------------------ our arm
    import torch
    import paper_2606_20519_b200 as hp

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    hp.load_library()
    hp.set_option("two_stage", args.two_stage)
    hp.set_option("two_stage_min_n", args.two_stage_min_n)
    jmax = 116

    def device_inputs(c):
        w = workloads.make(c)
        parts = [hp.pack(torch.from_numpy(np.ascontiguousarray(b.X.T)).to(dev)) for b in w.blocks]
        return w.sizes, torch.cat(parts)

    def count_pos(sizes, sv):
        out, off = [], 0
        for n in sizes:
            if n >= 2:
                lam = hp.eigvalsh(sv[off:off + n * n].clone(), n)
                out.append(int((lam > 0).sum().item()))
            else:
                out.append(int(n == 1 and sv[off].item() > 0))
            off += n * n
        return out

    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def time_device(sizes, sv, out, steps, warmup):
        for _ in range(warmup):
            hp.project_(sizes, sv, out)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        barrier()
        for a, b in ev:
            flush.zero_()                       # evict L2 between timed iterations
            a.record()
            hp.project_(sizes, sv, out)
            b.record()
        barrier()
        ms = [a.elapsed_time(b) for a, b in ev]
        return sum(ms), ms

    def time_e2e(sizes, h_in, h_out, steps, warmup):
        for _ in range(warmup):
            hp.project_host(sizes, h_in, h_out)
        barrier()
        tot = 0.0
        for _ in range(steps):
            flush.zero_()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            hp.project_host(sizes, h_in, h_out)   # H2D + projection + D2H + stream sync inside
            tot += time.perf_counter() - t0
        barrier()
        return tot * 1e3

    def max_over_ranks(x):
        if dist is None:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    sizes, sv = device_inputs(cfg)
    out = torch.empty_like(sv)
    kpos = count_pos(sizes, sv)
    K, W = max(args.steps, 1), args.warmup

    # FP64 peak of this GPU, measured here (MEASURED_PEAKS.json has no FP64 figure): DFMA and DMMA chains
    def probe(kind):
        best = 0.0
        for it in range(4):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fl = hp.fp64_peak_probe(kind, 4096)
            b.record()
            torch.cuda.synchronize()
            if it:
                best = max(best, fl / (a.elapsed_time(b) * 1e-3) / 1e12)
        return best
    peak_dfma, peak_dmma = probe(0), probe(1)
    fp64_peak = max(peak_dfma, peak_dmma)

    vis = os.environ.get("CUDA_VISIBLE_DEVICES", "").split(",")
    phys = int(vis[local_rank]) if local_rank < len(vis) and vis[local_rank].isdigit() else local_rank
    sampler = ClockSampler(phys)
    sampler.start()
    total_ms, per = time_device(sizes, sv, out, K, W)
    clocks = sampler.stop()
    launches_per_step = hp.last_launch_count()
    total_ms = max_over_ranks(total_ms)
    ms_per_step = total_ms / K
    value = world * 1.0 / (ms_per_step * 1e-3)      # cone-list projections per second, all replicas

    # stage timers: same K steps again with the library's CUDA-event spans on the launching stream
    def profile_stages(szs, v, o, reps):
        hp.set_option("profile", 1)
        acc_ms = {}
        for _ in range(reps):
            flush.zero_()
            hp.project_(szs, v, o)
            for name, (ms, spans) in hp.profile_read().items():
                a = acc_ms.setdefault(name, [0.0, 0])
                a[0] += ms; a[1] += spans
        hp.set_option("profile", 0)
        return {k: {"ms_per_step": x[0] / reps, "launch_spans_per_step": x[1] / reps} for k, x in acc_ms.items() if x[1]}

    hbm_peak, hbm_src = measured_hbm_gbs()
    fp64_src = (f"measured in this run by hpsd_fp64_peak_probe: DFMA {peak_dfma:.1f}, DMMA {peak_dmma:.1f} TFLOP/s "
                "(MEASURED_PEAKS.json has no FP64 figure)")

    def route_of(n):
        """The size class / reduction route the library's defaults (or --two-stage) give a block of size n."""
        if n <= 32:
            return "jacobi"
        if n <= jmax:
            return "medium"
        if args.two_stage == 1 and n >= 96 or args.two_stage == 2 and n >= args.two_stage_min_n:
            return "two_stage"
        return "cluster" if n <= 631 else "panel"

    def build_roofline(c, szs, kp, stages, ms_step):
        """Roofline object of the dominant stage of one workload."""
        dom = max(stages, key=lambda k: stages[k]["ms_per_step"])
        dom_ms = stages[dom]["ms_per_step"]
        dom_spans = max(stages[dom]["launch_spans_per_step"], 1)
        big = [n for n in szs if route_of(n) in ("cluster", "panel", "two_stage")]
        routes = sorted({route_of(n) for n in big})
        dom_flops = stage_flops(dom, szs, kp, route_of)
        F = sum(f_alg(n, k) for n, k in zip(szs, kp))
        tf = dom_flops / (dom_ms * 1e-3) / 1e12 if dom_ms > 0 else 0.0
        if dom == "S2S3_tridiag_panel" and routes == ["cluster"]:
            # matrix resident in the shared memory of one 16-CTA cluster: HBM sees the svec once (8 n^2 bytes) and the
            # reflectors once (~8 n^2 bytes); the bound is FP64 FMA issue (unblocked rank-2 update + mat-vec, DFMA)
            tr, trs = ncu_traffic("tridiag_cluster_kernel", c)
            rl = {"kernel": "tridiag_cluster_kernel (S1+S2+S3)", "bound": "alu", "achieved": tf, "peak": peak_dfma, "unit": "TFLOP/s",
                  "frac": tf / peak_dfma if peak_dfma else None, "traffic": tr, "traffic_source": trs,
                  "peak_source": fp64_src + "; DFMA figure, whole chip", "algorithmic_flops_per_step": dom_flops,
                  "algorithmic_bytes_per_step": sum(16.0 * n * n for n in big),
                  "regime": "latency-bound: one 16-CTA cluster, ~2 cluster exchanges + a scalar chain per column",
                  "sms_used": 16, "frac_of_16_sm_dfma_peak": tf / (peak_dfma * 16.0 / 148.0) if peak_dfma else None}
        elif dom == "S2S3_tridiag_panel" and "panel" in routes and max(big) > 1888:
            # streaming regime of the one-stage panel kernel: the stored lower triangle of the trailing matrix passes
            # through the SMs once per column: HBM/L2-bound by design
            dom_bytes = sum(panel_bytes(n) for n in big)
            gbs = dom_bytes / (dom_ms * 1e-3) / 1e9 if dom_ms > 0 else 0.0
            tr, trs = ncu_traffic("tridiag_panel_kernel", c)
            rl = {"kernel": "tridiag_panel_kernel (S2/S3 mat-vec half)", "bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s",
                  "frac": gbs / hbm_peak, "traffic": tr, "traffic_source": trs, "peak_source": hbm_src,
                  "regime": "streaming: trailing tiles do not fit the SMs' shared memory (n > 1888)",
                  "algorithmic_bytes_per_step": dom_bytes, "algorithmic_flops_per_step": dom_flops,
                  "flop_fraction_of_fp64_peak": tf / fp64_peak if fp64_peak else None}
        elif dom == "S2S3_tridiag_panel" and "panel" in routes:
            # resident regime: HBM sees one read per panel; the kernel is bound by two grid barriers and a scalar chain per column
            rl = {"kernel": "tridiag_panel_kernel (S2/S3 mat-vec half)", "bound": "alu", "achieved": tf, "peak": fp64_peak, "unit": "TFLOP/s",
                  "frac": tf / fp64_peak if fp64_peak else None, "traffic": None, "traffic_source": None, "peak_source": fp64_src,
                  "regime": "latency-bound: tiles resident in shared memory, 2 grid barriers per column (7-11 us per column)",
                  "algorithmic_flops_per_step": dom_flops}
        elif dom in ("S3_bulge_chasing", "S5_backtransform_q2"):
            vf = variant_flops(dom, szs, kp, route_of)
            vtf = vf / (dom_ms * 1e-3) / 1e12 if dom_ms > 0 else 0.0
            rl = {"kernel": dom, "bound": "alu" if dom == "S3_bulge_chasing" else "tensor", "achieved": vtf, "peak": fp64_peak, "unit": "TFLOP/s",
                  "frac": vtf / fp64_peak if fp64_peak else None, "traffic": None, "traffic_source": None, "peak_source": fp64_src,
                  "regime": "latency-bound chain of ~2n hops" if dom == "S3_bulge_chasing" else "DMMA tiles on diamond blocks",
                  "algorithmic_flops_per_step": 0.0, "variant_flops_per_step": vf,
                  "note": "extra work of the two-stage variant: not part of F_alg (SURVEY.md section 8(d))"}
        else:
            bound = "alu" if dom in ("S9_jacobi", "S10_householder_ql") else ("hbm" if dom == "S1_unpack" else "tensor")
            if bound == "hbm":
                dom_bytes = sum(16.0 * n * n for n in big)
                gbs = dom_bytes / (dom_ms * 1e-3) / 1e9 if dom_ms > 0 else 0.0
                rl = {"kernel": dom, "bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                      "traffic": None, "traffic_source": None, "peak_source": hbm_src, "algorithmic_bytes_per_step": dom_bytes}
            else:
                rl = {"kernel": dom, "bound": bound, "achieved": tf, "peak": fp64_peak, "unit": "TFLOP/s",
                      "frac": tf / fp64_peak if fp64_peak else None, "traffic": None, "traffic_source": None,
                      "peak_source": fp64_src, "algorithmic_flops_per_step": dom_flops}
        rl.update({
            "avg_launch_ms": dom_ms / dom_spans, "launches_per_step": dom_spans,
            "share_of_step": dom_ms / sum(x["ms_per_step"] for x in stages.values()),
            "fp64_peak_tflops": fp64_peak, "fp64_peak_source": fp64_src,
            "whole_path": {"f_alg_flops": F, "achieved_tflops": F / (ms_step * 1e-3) / 1e12,
                           "frac_of_fp64_peak": F / (ms_step * 1e-3) / 1e12 / fp64_peak if fp64_peak else None,
                           "hbm_floor_ms": 16.0 * sum(n * n for n in szs) / (hbm_peak * 1e9) * 1e3},
            "stages": stages,
        })
        return rl

    stages = profile_stages(sizes, sv, out, K)
    roofline = build_roofline(cfg, sizes, kpos, stages, ms_per_step)

    # end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    h_in = sv.cpu().pin_memory()
    h_out = torch.empty_like(h_in).pin_memory()
    e2e_ms = max_over_ranks(time_e2e(sizes, h_in, h_out, K, W)) / K
    e2e = {"value": world / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms,
           "h2d_bytes_per_step": int(sv.numel() * 8), "d2h_bytes_per_step": int(sv.numel() * 8)}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": wname, "sizes": sizes if len(sizes) <= 4 else f"{len(sizes)} blocks",
                   "positive_eigenvalues": kpos if len(kpos) <= 4 else None,
                   "l2": f"L2 flushed between timed iterations by writing a {L2_FLUSH_BYTES >> 20} MiB buffer",
                   "parallelism": "replicas only (a single block does not shard)" if world > 1 else "single GPU"},
        "ms_min": min(per), "ms_median": statistics.median(per),
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step * K, "launches_per_step": launches_per_step,
        "roofline": roofline,
    }

    if rank == 0 and world == 1:
        extra = {}
        # every other BASELINE.json config, same timing protocol (fewer steps), with its dominant stage and roofline:
        # the driver's record then carries all five workloads
        others = [] if args.no_secondary else [c for c in (1, 2, 4, 5) if c != cfg]
        if args.only_n4096:
            others = [5] if cfg != 5 else []
        cached = {cfg: (sizes, sv)}
        for c in others:
            s2, v2 = device_inputs(c)
            cached[c] = (s2, v2)
            o2 = torch.empty_like(v2)
            k2 = count_pos(s2, v2)
            steps2 = 3 if c in (4, 5) else 10
            t2, per2 = time_device(s2, v2, o2, steps2, 3)
            nl = hp.last_launch_count()
            st2 = profile_stages(s2, v2, o2, 2)
            r2 = build_roofline(c, s2, k2, st2, t2 / steps2)
            extra[f"cfg{c}"] = {"ms_per_call": t2 / steps2, "ms_min": min(per2), "launches": nl,
                                "f_alg_gflop": r2["whole_path"]["f_alg_flops"] / 1e9,
                                "frac_of_fp64_peak": r2["whole_path"]["frac_of_fp64_peak"],
                                "dominant_stage": {k: r2[k] for k in ("kernel", "bound", "achieved", "peak", "unit", "frac", "share_of_step", "regime") if k in r2},
                                "stages_ms": {k: round(x["ms_per_step"], 4) for k, x in st2.items()}}
            if c == 4:
                extra["cfg4"]["note"] = ("ms_per_call: the two large blocks run side by side (panel lanes); stages_ms / share_of_step: the "
                                         "library's stage timers, which run the blocks one after the other on one stream")
            del o2
        # one-stage (cluster / panel kernel) against the two-stage reduction (S2 dense -> band, S3 bulge chasing, Q2) on
        # the paper's large sizes: the measurement the default route rests on
        if not args.no_routes and not args.no_secondary:
            routes = {}
            blocks = {}
            if 3 in cached:
                blocks[625] = cached[3][1]
            if 4 in cached:
                v4 = cached[4][1]
                blocks[1296] = v4[:1296 * 1296]
                blocks[2401] = v4[1296 * 1296:1296 * 1296 + 2401 * 2401]
            if 5 in cached:
                blocks[4096] = cached[5][1]
            for n_, v_ in sorted(blocks.items()):
                v_ = v_.contiguous()
                o_ = torch.empty_like(v_)
                row = {}
                for mode, name in ((0, "one_stage"), (1, "two_stage")):
                    hp.set_option("two_stage", mode)
                    t_, per_ = time_device([n_], v_, o_, 3, 3)
                    st_ = profile_stages([n_], v_, o_, 1)
                    red = sum(x["ms_per_step"] for k_, x in st_.items() if k_ in ("S1_unpack", "S2S3_tridiag_panel", "S2_her2k_trailing", "S3_bulge_chasing"))
                    row[name] = {"ms_per_projection": t_ / 3, "reduction_S1_S2_S3_ms": red,
                                 "extra_backtransform_q2_ms": st_.get("S5_backtransform_q2", {}).get("ms_per_step", 0.0)}
                hp.set_option("two_stage", args.two_stage)
                row["default_route"] = "two_stage" if route_of(n_) == "two_stage" else "one_stage"
                routes[str(n_)] = row
                del o_
            line["reduction_routes"] = routes
        del cached
        if cfg == 3 and not args.no_secondary:
            # information only (the headline `value` stays one block per call): eight n=625 blocks in ONE call run on the
            # library's lane streams, one 16-CTA cluster each
            s8, v8 = sizes * 8, sv.repeat(8)
            o8 = torch.empty_like(v8)
            t8, per8 = time_device(s8, v8, o8, 5, 3)
            line["batched_call"] = {"blocks_per_call": 8, "ms_per_call": t8 / 5, "projections_per_s": 8.0 / (t8 / 5 * 1e-3),
                                    "note": "eight n=625 blocks in one hpsd_project call (lanes); not the headline metric"}
            del v8, o8
        # NEXT-3: the affine-projection step z_x = (a_x - A^T a_y)/2, z_y = a_y + A z_x on the device,
        # d = 5 (n = 625) and d = 8 (n = 4096); HBM-bound streaming passes (information only, not the headline metric)
        if not args.no_secondary:
            aff = {}
            for d_ in (5, 8):
                af = hp.Affine(d_)
                g_ = torch.Generator(device=dev); g_.manual_seed(20519 + d_)
                ax = torch.randn(af.m, dtype=torch.float64, device=dev, generator=g_)
                ay = torch.randn(af.n * af.n, dtype=torch.float64, device=dev, generator=g_)
                zx, zy = torch.empty_like(ax), torch.empty_like(ay)
                for _ in range(3):
                    af.project_(ax, ay, zx, zy)
                evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(10)]
                for a_, b_ in evs:
                    flush.zero_()
                    a_.record(); af.project_(ax, ay, zx, zy); b_.record()
                torch.cuda.synchronize()
                ms_ = statistics.median(a_.elapsed_time(b_) for a_, b_ in evs)
                alg_bytes = 16.0 * af.n * af.n + 16.0 * af.m            # a_y in, z_y out, a_x in, z_x out
                moved = 312.0 * af.n * af.n     # the 12 streaming passes of affine.cu: 24 + 4 x 32 (A^T), 8 + 24 + 3 x 32 + 32 (A) bytes per n^2
                aff[f"d{d_}"] = {"n": af.n, "m": af.m, "ms": ms_, "launches": hp.last_launch_count(),
                                 "algorithmic_gbs": alg_bytes / (ms_ * 1e-3) / 1e9, "moved_gbs_estimate": moved / (ms_ * 1e-3) / 1e9,
                                 "hbm_peak_gbs": hbm_peak}
                af.destroy()
                del ax, ay, zx, zy
            line["affine_step"] = aff
        # host cost of one call through the explicit plan handle: config 1 (one n = 16 block), enqueue only,
        # no synchronisation inside the loop; the plan replays its CUDA graph from the third call on
        if not args.no_secondary:
            s1, v1 = device_inputs(1)
            o1 = torch.empty_like(v1)
            pl1 = hp.Plan(s1)
            for _ in range(5):
                pl1.project_(v1, o1)
            torch.cuda.synchronize()
            # bursts of 16 calls, synchronised (untimed) in between: a long back-to-back run fills the launch queue and would
            # measure the GPU's time per call instead of the host's
            reps, t_enq = 0, 0.0
            for _ in range(64):
                t0 = time.perf_counter()
                for _ in range(16):
                    pl1.project_(v1, o1)
                t_enq += time.perf_counter() - t0
                reps += 16
                torch.cuda.synchronize()
            t_enq /= reps
            t0 = time.perf_counter()
            for _ in range(2000):
                pl1.project_(v1, o1)
            torch.cuda.synchronize()
            t_all = (time.perf_counter() - t0) / 2000
            c_us = pl1.host_overhead_us(v1, o1, 2000)
            pl1.destroy()
            line["plan_host_overhead"] = {"workload": "cfg1 (1 x n=16), hpsd_plan_project, CUDA graph warm, enqueue only",
                                          "c_abi_enqueue_us_per_call": c_us,
                                          "python_binding_enqueue_us_per_call": t_enq * 1e6, "throughput_us_per_call_2000_back_to_back": t_all * 1e6,
                                          "note": "enqueue figures: bursts of 16 calls with an untimed synchronisation in between (a full launch queue would "
                                                  "show the GPU's time per call); c_abi: loop inside the library (hpsd_plan_host_overhead); the Python "
                                                  "figure adds ctypes/torch marshalling; throughput: 2000 calls back to back including the final synchronise"}
        # NEXT-1: the same projection on complex64 STORAGE (FP32 svecs in HBM, FP64 arithmetic): configs 3 and 2
        if not args.no_secondary:
            c64 = {}
            for c in (3, 2):
                sc, vc = device_inputs(c)
                v32 = vc.float()
                o32 = torch.empty_like(v32)
                tot, _ = time_device(sc, v32, o32, 10, 3)
                c64["cfg%d" % c] = {"ms_per_call": tot / 10, "svec_bytes_per_call": 2 * 4 * int(v32.numel())}
                del v32, o32, vc
            c64["note"] = ("hpsd_project_c64: FP32 svecs, every load widened and every store rounded, the FP64 kernels in between; "
                           "FP32 arithmetic is not built (DESIGN.md section 10)")
            line["c64_storage"] = c64
        line["other_configs"] = extra
        if "cfg5" in extra:
            line["ms_per_projection_n4096"] = extra["cfg5"]["ms_per_call"]
        if not args.no_cpu_baseline:
            v, per_step, threads, sample = run_oracle(cfg, 1, 0, min_seconds=10.0)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                                    "ms_per_projection": per_step * 1e3}
        line["paper_context"] = ("paper (Tesla T4, JAX eigh only, complex128): 0.06 s at n=625, 6.33 s at n=4096 "
                                 "(PAPER.md:1515-1518); whole SDP six-fold vs CPU SCS (PAPER.md:1554); other hardware, context only")
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
