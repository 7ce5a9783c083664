#!/usr/bin/env python
"""bench.py -- throughput of the LArTPC charge hot path (arXiv 2212.09807) on B200.

One "step" = one pass of the whole hot path (S1 quench .. S6 electronics, `lartpc_run_spill`) over one
synthetic spill.  Metric (BASELINE.json): segments/s (whole job) with ms/spill as `ms_per_step`.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]
  python bench.py --config 4            BASELINE configs[4]: the induced-current sweep (S4 + S5 only), one JSON line
  python bench.py --light [--config k]  the light simulation on that config's segments, one JSON line

* `value`     segments/s with the segment arrays already resident in HBM (device-timed, CUDA events).
* `e2e`       same metric through the C-ABI with HOST (pinned) segment arrays: host->device copy of the nine
              float32 arrays and device->host read of the hit list inside the timed region.
* `roofline`  the dominant kernel (the S4 response on the tcgen05 tensor cores): multiply-adds the method needs for the
              charge it found (counted on the device) x 2 / its CUDA-event time, against the measured bf16 / fp16 tensor
              peak of MEASURED_PEAKS.json (sustained figure when the step is longer than 50 ms, else the burst figure); `executed_*` = the dense MMA
              work actually issued (device-counted tcgen05.mma instructions); `traffic` = its DRAM bytes per launch.
* `rooflines` one entry per kernel of the path: S1, S2, S3, S5, S6 against the measured HBM copy bandwidth (algorithmic bytes
              of SURVEY.md 8(d) and the bytes the kernel moves), the charge lattice against the SM's thread-instruction
              rate, the response against the tensor peak (DESIGN.md section 5 has every per-unit figure).
* `cpu_baseline`  the fp64 oracle (oracle/, as it stands) on this host's cores, on a bounded sample: all cores, and one core.
* `--impl reference`  times that oracle alone (there is no reference code for this paper).
N > 1 (torchrun): every rank simulates its own independent spill (seed + rank), no data-path collective;
`value` sums the ranks' segments over the max-over-ranks time ("scaling": "weak").
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

from paper_2212_09807_b200 import workloads  # noqa: E402

METRIC = "segments/s (ms/spill in ms_per_step)"
WORKLOAD_NAMES = {
    0: "configs[0] PR1 single MIP muon, 100 segments, 32x32 pixels",
    1: "configs[1] cosmic muons, one TPC, 70x70 pixels, 30 cm drift",
    2: "configs[2] neutrino-like interactions, 2x2 modules (8 TPCs), ~1e5 segments",
    3: "configs[3] full ND-LAr-scale beam spill, 70 TPCs, ~1.07e7 pixels, ~5e6 segments",
}


# DRAM bytes per spill of the tensor-core response measured with ncu on the benched workload and launch configuration
# (profiles/r2_traffic_c3.md: dram__bytes_read.sum + dram__bytes_write.sum over the 4 launches of one configs[3] spill),
# keyed by (config, n_segments, n_tiles); any other workload reports the byte model of the plan instead and says so
MEASURED_RESPONSE_TRAFFIC = {(3, 4805366, 3113102): 62959459328.0 + 82048449024.0}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[0, 1, 2, 3, 4],
                    help="0-3: one spill of that BASELINE config; 4: the induced-current sweep (S4 + S5 only, one axis at a time)")
    ap.add_argument("--sweep-max-segments", type=int, default=10_000_000, help="largest segment count of the config-4 sweep")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--segments", type=int, default=None, help="override the segment target of configs 2/3")
    ap.add_argument("--response", default="auto", choices=["auto", "tensor", "ffma"],
                    help="S4 response path: tcgen05 tensor cores or the FP32-pipe FFMA2 kernel")
    ap.add_argument("--light", action="store_true",
                    help="time the light simulation (SURVEY 8(f) NEXT-3, eqs. 4.1-4.6) on the chosen config's segments instead")
    ap.add_argument("--light-sensors", type=int, default=None, help="photosensors of the --light run (default 64 at config 3, else 16)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-sample", type=int, default=1000, help="segments in the oracle's bounded sample")
    return ap.parse_args()


def make_workload(cfg: int, rank: int, segments=None):
    kw = {}
    if segments is not None and cfg in (2, 3):
        kw["target"] = segments
    if rank:
        kw["seed"] = workloads.SEED_BASE + cfg + 1000 * rank
    return workloads.make_config(cfg, **kw)


# --------------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md "clocks line")
# --------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap,power.limit")

    def __init__(self, index: int):
        self.index, self.rows, self._stop, self._t = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5)
                if out.returncode == 0 and out.stdout.strip():
                    self.rows.append([c.strip() for c in out.stdout.strip().splitlines()[0].split(",")])
            except Exception:
                pass
            self._stop.wait(0.1)

    def start(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()

    def stop(self):
        self._stop.set()
        if self._t:
            self._t.join(timeout=6)
        sm, mx, pw, lim, reasons = [], [], [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            try:
                pw.append(float(r[2])); lim.append(float(r[7]))
            except Exception:
                pass
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm),
                "power_w": float(np.median(pw)) if pw else None, "power_limit_w": max(lim) if lim else None}


# --------------------------------------------------------------------------------------------------
# the oracle on the host cores (cpu_baseline leg and --impl reference)
# --------------------------------------------------------------------------------------------------
def oracle_sample(wl, n_sample: int):
    """A contiguous block of segments from the middle of the spill (one shower / track neighbourhood)."""
    n = wl.n_segments
    m = min(n_sample, n)
    lo = max(0, n // 2 - m // 2)
    return wl.subset(np.arange(lo, lo + m)), "segments [%d, %d) of %d, all pixels they reach, full chain O1-O6" % (
        lo, lo + m, n)


def time_oracle(wl, n_sample: int, cores=None):
    import oracle
    oracle.build()
    sub, what = oracle_sample(wl, n_sample)
    cores = (os.cpu_count() or 1) if cores is None else cores
    t0 = time.perf_counter()
    res = oracle.run_chain(sub, threads=cores)
    dt = time.perf_counter() - t0
    return {"value": sub.n_segments / dt, "unit": "segments/s", "cores": cores, "kind": "oracle",
            "sample": what + " (%.1f s, %d hits)" % (dt, len(res["hit_pixel"]))}, dt, sub.n_segments


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step = one bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = make_workload(args.config, 0, args.segments)
    n_sample = max(50, args.cpu_sample // 4)            # sized so steps + warm-up end within a few minutes
    total, segs, info = 0.0, 0, None
    for i in range(args.warmup + args.steps):
        if i >= min(args.warmup, 1) and i < args.warmup:
            continue                                      # one warm-up pass is enough for a CPU program
        info, dt, ns = time_oracle(wl, n_sample)
        if i >= args.warmup:
            total += dt
            segs += ns
    value = segs / total
    info["value"] = value
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": "segments/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_NAMES[args.config], "n_segments": wl.n_segments,
                       "n_pixels": wl.n_pixels, "step": "oracle O1-O6 on a bounded sample: " + info["sample"]},
            "cpu_baseline": info,
            "e2e": {"value": value, "unit": "segments/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def reduce_over_ranks(ms: float, n_segments: int, world: int, device):
    """Whole-job figures of a weak-scaling run (every rank simulates its own spill, no data-path collective): the time is
    the MAX over ranks, the work the SUM of the ranks' segments."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    nseg = torch.tensor([float(n_segments)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(nseg, op=dist.ReduceOp.SUM)
    return float(t.item()), float(nseg.item())


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2212_09807_b200 import lartpc

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a B200: the LArTPC path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    wl = make_workload(args.config, rank, args.segments)
    n = wl.n_segments
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut, device="cuda:%d" % local, response=args.response)
    if wl.disabled_pixels is not None:
        sim.set_disabled_pixels(wl.disabled_pixels)
    host = {k: torch.from_numpy(np.ascontiguousarray(wl.segments[k], dtype=np.float32)).pin_memory()
            for k in workloads.SEG_FIELDS}
    seg = {k: v.to(dev) for k, v in host.items()}
    ws = torch.empty(sim.workspace_bytes(n), dtype=torch.uint8, device=dev)
    hit_cap = int(min(64_000_000, max(1 << 16, 8 * n)))
    hits, st = sim.run_spill(seg, wl.seed, hit_cap, workspace=ws)           # sizes the library's plan buffers
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)           # > 126 MB L2

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing -------------------------------------------------------------------
    for _ in range(args.warmup):
        flush.zero_()
        hits, st = sim.run_spill(seg, wl.seed, hit_cap, workspace=ws, hits=hits)
    peak_scalar, peak_packed = lartpc.measure_fp32_peak(0), lartpc.measure_fp32_peak(1)
    sim.set_profiling(True)
    launches0 = lartpc.kernel_launches()
    stage_ms = {k: [] for k in sim.STAGES}
    stage_n = {k: 0 for k in sim.STAGES}
    cnt = {k: 0.0 for k in sim.COUNTERS}
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    clocks = ClockSampler(local)
    barrier()
    clocks.start()
    for i in range(args.steps):
        flush.zero_()
        ev[i][0].record()
        hits, st = sim.run_spill(seg, wl.seed, hit_cap, workspace=ws, hits=hits)
        ev[i][1].record()
        ms, ln, _ = sim.stage_ms()
        for k in sim.STAGES:
            stage_ms[k].append(ms[k])
            stage_n[k] += ln[k]
        for k, v in sim.counters().items():
            cnt[k] += v / args.steps
    barrier()
    clk = clocks.stop()
    launches = lartpc.kernel_launches() - launches0
    sim.set_profiling(False)
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = sum(step_ms)
    total_ms_max, n_all = reduce_over_ranks(total_ms, n, world, dev)
    median_ms, _ = reduce_over_ranks(float(np.median(step_ms)), n, world, dev)

    # ---- end to end through the C-ABI with host buffers ------------------------------------------
    # a user's loop: pinned host segment arrays in, pinned host hit arrays out, device buffers allocated once; one untimed
    # pass first (pinned-buffer and allocator warm-up), then the timed passes with both copies inside
    e2e_ev = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
    dseg = {k: torch.empty_like(v) for k, v in seg.items()}
    n_out = int(st.n_hits * 1.25) + 4096
    hout = {k: torch.empty(n_out, dtype=torch.int32).pin_memory() for k in ("hit_pixel", "hit_tick", "hit_adc")}
    d2h = 0

    def e2e_step():
        for k, v in host.items():
            dseg[k].copy_(v, non_blocking=True)
        h, st2 = sim.run_spill(dseg, wl.seed, hit_cap, workspace=ws, hits=hits)
        nh = min(int(st2.n_hits), n_out)
        for k in hout:
            hout[k][:nh].copy_(h[k][:nh], non_blocking=True)
        torch.cuda.synchronize()                                     # the hit list is in host memory
        return 3 * 4 * nh + 32

    e2e_step()
    barrier()
    e2e_ev[0].record()
    for i in range(args.steps):
        flush.zero_()
        d2h = e2e_step()
    e2e_ev[1].record()
    barrier()
    flush_ms = 0.0
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record()
    for i in range(args.steps):
        flush.zero_()
    f1.record()
    torch.cuda.synchronize()
    flush_ms = f0.elapsed_time(f1)
    e2e_ms, _ = reduce_over_ranks(e2e_ev[0].elapsed_time(e2e_ev[1]) - flush_ms, n, world, dev)

    if rank == 0:
        mp = {}
        try:
            mp = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        hbm_peak = float(mp.get("hbm_gbs", 6650.0))
        hbm_src = "MEASURED_PEAKS.json hbm_gbs (measured copy)" if mp.get("hbm_gbs") else "fallback of B200_PROFILING.md"
        per_step = {k: float(np.median(v)) for k, v in stage_ms.items()}          # ms per step, median over the steps
        n_launch = {k: stage_n[k] / args.steps for k in sim.STAGES}
        P = wl.params
        K, nb2, ww = int(P["lut_ticks"]), int(P["bins_per_pixel"]) ** 2, int(P["window_pixels"]) ** 2
        n_tiles, n_pairs, n_act, n_samp, n_hits = (int(st.n_tiles), int(st.n_pairs), int(st.n_active_pixels),
                                                   int(st.total_samples), int(st.n_hits))
        sm_hz = 1e6 * float(clk["sm_mhz"] or 1965.0)

        def hbm_entry(stage, kernel, alg_bytes, moved_bytes, note):
            t = per_step[stage] * 1e-3
            return {"kernel": kernel, "stage": stage, "bound": "hbm", "unit": "GB/s", "peak": hbm_peak, "peak_source": hbm_src,
                    "achieved": alg_bytes / t / 1e9 if t > 0 else None, "frac": alg_bytes / t / 1e9 / hbm_peak if t > 0 else None,
                    "moved_gbs": moved_bytes / t / 1e9 if t > 0 else None,
                    "moved_frac": moved_bytes / t / 1e9 / hbm_peak if t > 0 else None,
                    "algorithmic_bytes_per_step": alg_bytes, "moved_bytes_per_step": moved_bytes,
                    "ms_per_step": per_step[stage], "launches_per_step": n_launch[stage], "note": note}

        rooflines = [
            hbm_entry("quench", "quench_kernel (S1)", 44.0 * n, 36.0 * n,
                      "algorithmic 36 B in + 8 B out per segment (SURVEY 8(d)); the kernel reads 7 of the 9 arrays"),
            hbm_entry("drift", "drift_kernel (S2)", 80.0 * n, 100.0 * n,
                      "algorithmic ~80 B per segment (SURVEY 8(d)); moved 32 B in + 4 B n_e + 64 B out (float64 end points)"),
            hbm_entry("pixels_from_segments", "pixmap_kernel + tile plan (S3)", 64.0 * n,
                      (44.0 + 56.0 + 96.0 + 40.0) * n + 16.0 * n_pairs + 120.0 * n_tiles,
                      "algorithmic 64 B per segment (SURVEY 8(d)); moved (estimate from the kernels' accesses): boxes, 96 B record "
                      "per segment, 4 B per (segment, charged pixel) pair written + sorted, tile descriptors / lists / slots"),
        ]
        # S4 charge lattice: thread-instruction rate of the SMs (the kernel is bound by issue slots: erf, products, splits)
        t_ch = per_step["induced_current_charge"] * 1e-3
        OPS_PER_COLUMN = 87 * 13 + 164 + 150      # 87 erf x 13 instructions, 164 products, 150 split / convert / store
        alu_peak = sim_sm_count(torch, local) * 128 * sm_hz / 1e12                 # T thread-instructions / s (all four schedulers issuing)
        ch_ops = cnt["charge_columns"] * OPS_PER_COLUMN
        rooflines.append({"kernel": "charge_lattice_tc_kernel (S4a: charge per LUT cell, tcgen05 + erf weights)",
                          "stage": "induced_current_charge", "bound": "alu", "unit": "T thread-instructions/s",
                          "achieved": ch_ops / t_ch / 1e12 if t_ch > 0 else None, "peak": alu_peak,
                          "frac": ch_ops / t_ch / 1e12 / alu_peak if t_ch > 0 else None,
                          "peak_source": "SMs x 128 lanes x SM clock sampled during the run (one instruction per lane per cycle)",
                          "operand_columns_per_step": cnt["charge_columns"], "instructions_per_column": OPS_PER_COLUMN,
                          "tensor_tflops": cnt["charge_mma"] * 2.0 * 128 * 64 * 16 / t_ch / 1e12 if t_ch > 0 else None,
                          "ms_per_step": per_step["induced_current_charge"],
                          "launches_per_step": n_launch["induced_current_charge"],
                          "note": "operand columns (rule nodes / sample points x tiles) counted on the device x instructions one "
                                  "column costs (its weights: 87 erf, 164 products, fp16 splits and stores)"})
        n_resp = max(stage_n["induced_current_response"], 1)
        s4_ms = sum(stage_ms["induced_current_response"]) / n_resp
        t_rs = per_step["induced_current_response"] * 1e-3
        fma_per_launch = cnt["fma_needed"] * args.steps / n_resp
        useful = 2.0 * fma_per_launch / (s4_ms * 1e-3) / 1e12 if s4_ms > 0 else 0.0
        if sim.response_mode == "tensor":
            # dense fp16 contraction on tcgen05: peak = measured bf16 GEMM peak (fp16 runs at the same rate)
            # timed inside a long step (> 50 ms of back-to-back kernels under the power cap): the sustained figure; else burst
            long_launch = sum(per_step.values()) > 50.0
            if mp.get("bf16_tflops"):
                peak = float(mp["bf16_tflops_sustained"] if long_launch and mp.get("bf16_tflops_sustained")
                             else mp["bf16_tflops"])
                peak_src = "MEASURED_PEAKS.json bf16 cuBLAS GEMM, %s figure (fp16 = bf16 rate)" % (
                    "sustained" if long_launch else "burst")
            else:
                peak, peak_src = 1590.0, "fallback of B200_PROFILING.md (MEASURED_PEAKS.json absent)"
            kq = K if (K + 15 + 15) // 16 * 16 <= 224 else 200               # LUT pieces of the tensor path
            nbw, rows = (kq + 15 + 15) // 16 * 16, ww * ((K + kq - 1) // kq)
            # every tcgen05.mma of the response (fp16, K = 16, or fp8, K = 32) occupies the pipe like 128 x NBW x 16 fp16
            # multiply-adds: fp16-equivalent flops of the instructions the kernel counted as it issued them
            executed = cnt["response_mma"] * 2.0 * 128 * nbw * 16 * args.steps / n_resp
            lut_bytes = rows * nb2 * nbw * 64.0
            partial_bytes = 4.0 * n_tiles * rows * (((64 + kq - 1 + 7) // 8) * 8)
            gen_bytes = cnt["response_items"] * nb2 * nbw * 64.0
            a_once = max(cnt["response_bytes_to_smem"] - gen_bytes, 0.0) / rows      # every charge block is copied once per target row
            dram = (a_once + partial_bytes + lut_bytes * n_launch["induced_current_response"]) / max(n_launch["induced_current_response"], 1)
            roof = {"kernel": "rtc::response_tc_kernel (S4b: induced current, response on tcgen05)", "bound": "tensor",
                    "achieved": useful, "peak": peak, "unit": "TFLOP/s", "frac": useful / peak,
                    "achieved_note": "algorithmic: non-zero charge cells x in-plane targets x lut_ticks x 2 (counted on "
                                     "the device), what the method needs whatever the decomposition",
                    "executed_tflops": executed / (s4_ms * 1e-3) / 1e12 if s4_ms > 0 else 0.0,
                    "executed_frac": executed / (s4_ms * 1e-3) / 1e12 / peak if s4_ms > 0 else None,
                    "executed_note": "tcgen05.mma instructions counted by the kernel as it issues them x 128 x NBW x 16 x 2 "
                                     "(an fp8 K = 32 instruction occupies the pipe like an fp16 K = 16 one)",
                    "smem_fill_gbs": cnt["response_bytes_to_smem"] / t_rs / 1e9 if t_rs > 0 else None,
                    "fp32_alu_peak": max(peak_scalar, peak_packed), "peak_source": peak_src,
                    "traffic": None, "traffic_model": dram,
                    "traffic_note": "traffic: dram__bytes_read.sum + dram__bytes_write.sum per launch from the ncu capture "
                                    "of this workload (profiles/r2_traffic_c3.md), null for a workload without one; "
                                    "traffic_model: bytes per launch from the plan and the kernel's counters (charged "
                                    "operand blocks read once, partial rows written, LUT image once): 0.80 of the measured "
                                    "figure at configs[3]"}
            meas = MEASURED_RESPONSE_TRAFFIC.get((args.config, int(n), int(n_tiles)))
            if meas is not None:
                roof["traffic"] = meas / max(n_launch["induced_current_response"], 1)
        else:
            peak = max(peak_scalar, peak_packed)
            roof = {"kernel": "response_kernel (S4 induced current, response on the FP32 pipe)", "bound": "alu",
                    "achieved": useful, "peak": peak, "unit": "TFLOP/s", "frac": useful / peak if peak else None,
                    "peak_source": "lartpc_measure_fp32_peak on this GPU (scalar FFMA %.1f, packed FFMA2 %.1f)"
                                   % (peak_scalar, peak_packed), "traffic": None}
            partial_bytes = 4.0 * n_tiles * ww * 266
        roof.update(launch_ms=s4_ms, flops_per_launch=2.0 * fma_per_launch, ms_per_step=per_step["induced_current_response"],
                    launches_per_step=n_launch["induced_current_response"], stage="induced_current_response",
                    share_of_step=per_step["induced_current_response"] / max(sum(per_step.values()), 1e-9))
        rooflines.append(dict(roof))
        rooflines.append(hbm_entry("sum_pixel_signals", "sum_pixel_kernel (S5)", 8.0 * n_samp, 0.87 * partial_bytes + 4.0 * n_samp,
                                   "algorithmic 4 B in + 4 B out per stored waveform sample; moved (estimate): the charged part "
                                   "(~87 %) of every tile's partial rows read once + the samples written"))
        rooflines.append(hbm_entry("electronics", "electronics_warp_kernel + hit compaction (S6)", 4.0 * n_samp + 12.0 * n_hits,
                                   4.0 * n_samp + 12.0 * n_hits + (4.0 * int(P["max_hits_per_pixel"]) + 24.0) * n_act,
                                   "algorithmic 4 B in per sample + 12 B per hit (SURVEY 8(d)); moved adds the per-pixel hit slots"))
        line = {
            "metric": METRIC, "value": n_all / (median_ms * 1e-3), "unit": "segments/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": median_ms,
            "ms_per_step_mean": total_ms_max / args.steps, "step_ms": step_ms,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": ("fp16 hi+lo operand splits with the cross terms in fp8 (e4m3), fp32 accumulate (S4 on tcgen05); fp32 "
                      "elsewhere, fp64 where an integer is decided" if sim.response_mode == "tensor" else
                      "f32 (S4 on the FP32 pipe), fp64 where an integer is decided"),
            "data": "synthetic",
            "config": {"workload": WORKLOAD_NAMES[args.config], "n_segments": n, "n_pixels": wl.n_pixels,
                       "n_readout_ticks": int(wl.params["n_readout_ticks"]), "n_tpcs": len(wl.tpcs),
                       "seed": wl.seed, "l2": "256 MiB flush write between timed steps",
                       "timing": "CUDA events per step on the launching stream; value from the median step",
                       "parallelism": "independent spill per GPU" if world > 1 else "single GPU",
                       "input_sha256": {k: v[:16] for k, v in wl.sha256().items()}},
            "stats": {"n_tiles": n_tiles, "n_pairs": n_pairs, "n_active_pixels": n_act,
                      "total_samples": n_samp, "n_hits": n_hits,
                      "n_hits_dropped": int(st.n_hits_dropped), "n_batches": int(st.n_batches)},
            "counters_per_step": cnt,
            "stage_ms_per_step": per_step,
            "e2e": {"value": n_all * args.steps / (e2e_ms * 1e-3), "unit": "segments/s",
                    "h2d_bytes_per_step": 9 * 4 * n, "d2h_bytes_per_step": int(d2h), "ms_per_step": e2e_ms / args.steps},
            "gpu_launches": int(launches),
            "clocks": clk,
            "roofline": roof,
            "rooflines": rooflines,
            "response_mode": sim.response_mode,
        }
        if not args.no_cpu_baseline and world == 1:
            base, _, _ = time_oracle(wl, args.cpu_sample)
            one, _, _ = time_oracle(wl, max(40, args.cpu_sample // 10), cores=1)
            base["one_core"] = one
            line["cpu_baseline"] = base
        print(json.dumps(line))
    sim.close()
    if world > 1:
        dist.destroy_process_group()


def sim_sm_count(torch, index):
    return int(torch.cuda.get_device_properties(index).multi_processor_count)


# --------------------------------------------------------------------------------------------------
# BASELINE configs[4]: induced-current kernel sweep (S4 charge lattice + S4 response + S5 sum), one axis at a time
# about the base point (1e5 segments of 1 mm at 30 cm drift, 5x5 window, K = 200), track-like placement on one plane
# --------------------------------------------------------------------------------------------------
SWEEP_BASE = dict(n_segments=100_000, seg_len_cm=0.1, drift_cm=30.0, window_pixels=5, lut_ticks=200)


def sweep_points(max_segments):
    pts = [("base", {})]
    pts += [("count", dict(n_segments=n)) for n in (1_000, 10_000, 1_000_000, 10_000_000) if n <= max_segments]
    pts += [("length", dict(seg_len_cm=l)) for l in (0.05, 0.2, 0.5, 1.0)]
    pts += [("drift", dict(drift_cm=d)) for d in (0.0, 1.0, 10.0, 50.0)]
    pts += [("window", dict(window_pixels=9))]
    pts += [("lut_ticks", dict(lut_ticks=k)) for k in (500, 1000, 2000)]
    return pts


def run_sweep(args):
    import torch
    from paper_2212_09807_b200 import lartpc
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a B200: the LArTPC path has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    hbm_peak = 6541.1
    try:
        hbm_peak = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
    except Exception:
        pass
    fp32_peak = max(lartpc.measure_fp32_peak(0), lartpc.measure_fp32_peak(1))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    rows, launches0 = [], lartpc.kernel_launches()
    clocks = ClockSampler(0)
    clocks.start()
    for axis, over in sweep_points(args.sweep_max_segments):
        kw = dict(SWEEP_BASE, **over)
        wl = workloads.make_config(4, **kw)
        n = wl.n_segments
        sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut, device="cuda:0", response=args.response)
        seg = sim.upload_segments(wl.segments)
        _, ne = sim.quench(seg)                                      # staged S1-S3 once: the tile geometry of this sim
        dr = sim.drift(seg, ne)
        _, pinfo = sim.pixels_from_segments(seg, dr)
        tile_bytes = 4.0 * pinfo.tile_charge_floats + 4.0 * pinfo.tile_targets * pinfo.tile_ticks
        del dr, ne
        free, _ = torch.cuda.mem_get_info()
        # longer segments and wider windows need more tile memory per segment than the library's 1 mm estimate
        ws = torch.empty(int(min(max(sim.workspace_bytes(n), 64 << 30), 0.8 * free)), dtype=torch.uint8, device=dev)
        hit_cap = int(min(64_000_000, max(1 << 16, 8 * n)))
        hits, st = sim.run_spill(seg, wl.seed, hit_cap, workspace=ws)
        for _ in range(max(args.warmup - 1, 0)):
            flush.zero_()
            hits, st = sim.run_spill(seg, wl.seed, hit_cap, workspace=ws, hits=hits)
        sim.set_profiling(True)
        acc = {k: 0.0 for k in sim.STAGES}
        fma = 0.0
        for _ in range(args.steps):
            flush.zero_()
            hits, st = sim.run_spill(seg, wl.seed, hit_cap, workspace=ws, hits=hits)
            ms, _, f = sim.stage_ms()
            for k in sim.STAGES:
                acc[k] += ms[k] / args.steps
            fma += f / args.steps
        t_ch, t_rs, t_sum = acc["induced_current_charge"], acc["induced_current_response"], acc["sum_pixel_signals"]
        t = t_ch + t_rs + t_sum
        # algorithmic HBM bytes of S4 + S5: 48 B / segment in, every stored waveform sample written once (4 B); the
        # tile intermediates (charge image + partial rows, written once and read once) are the decomposition's own
        inter = 2.0 * int(st.n_tiles) * tile_bytes
        alg = 48.0 * n + 4.0 * int(st.total_samples)
        rows.append(dict(axis=axis, **kw, n_segments_actual=n, response_mode=sim.response_mode,
                         n_tiles=int(st.n_tiles), n_active_pixels=int(st.n_active_pixels),
                         ms_charge=t_ch, ms_response=t_rs, ms_sum=t_sum, ms_s4_s5=t,
                         segments_per_s=n / (t * 1e-3) if t > 0 else None,
                         useful_tflops=2.0 * fma / ((t_ch + t_rs) * 1e-3) / 1e12 if t_ch + t_rs > 0 else None,
                         frac_fp32_peak=2.0 * fma / ((t_ch + t_rs) * 1e-3) / 1e12 / fp32_peak if t_ch + t_rs > 0 else None,
                         hbm_gbs_algorithmic=alg / (t * 1e-3) / 1e9 if t > 0 else None,
                         hbm_gbs_with_tile_intermediates=(alg + inter) / (t * 1e-3) / 1e9 if t > 0 else None,
                         frac_hbm_peak_with_intermediates=(alg + inter) / (t * 1e-3) / 1e9 / hbm_peak if t > 0 else None))
        sys.stderr.write("sweep %-9s %s: %d segments, %d tiles, S4+S5 %.2f ms (%s)\n"
                         % (axis, over, n, int(st.n_tiles), t, sim.response_mode))
        sim.close()
        del ws, seg, hits
        torch.cuda.empty_cache()
    clk = clocks.stop()
    base = rows[0]
    line = {"metric": "segments/s through S4 + S5 (induced current + per-pixel sum), configs[4] base point",
            "value": base["segments_per_s"], "unit": "segments/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": base["ms_s4_s5"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "fp16 hi+lo / fp8 (e4m3) cross terms, fp32 accumulate (S4 on tcgen05)", "data": "synthetic",
            "config": {"workload": "configs[4] induced-current sweep, one 226x677 plane, track-like placement",
                       "base": SWEEP_BASE, "l2": "256 MiB flush write between timed steps"},
            "fp32_alu_peak_tflops": fp32_peak, "hbm_peak_gbs": hbm_peak, "clocks": clk,
            "gpu_launches": int(lartpc.kernel_launches() - launches0), "sweep": rows}
    print(json.dumps(line))


def run_light(args):
    """Light simulation (NEXT-3) on the segments of configs[0..3]: S1 (recombination, shared with the charge path) and
    L1-L5 per step; stage times from the staged calls, step time from lartpc_light_run; one JSON line."""
    import torch
    from paper_2212_09807_b200 import lartpc
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a B200: the light path has no CPU fallback")
    dev = torch.device("cuda", 0)
    wl = make_workload(args.config, 0, args.segments)
    n = wl.n_segments
    n_det = args.light_sensors or (64 if args.config == 3 else 16)
    ls = workloads.light_setup(wl, n_det=n_det, vox_cm=8.0 if args.config == 3 else 4.0, noise=True)
    lp = ls.params
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    light = lartpc.LightSim(lp, ls.eff, ls.gain, ls.vis, ls.tprof, ls.resp, ls.noise_amp, ls.noise_k)
    host = {k: torch.from_numpy(np.ascontiguousarray(wl.segments[k], dtype=np.float32)).pin_memory() for k in workloads.SEG_FIELDS}
    seg = {k: v.to(dev) for k, v in host.items()}
    ws = torch.empty(light.workspace_bytes(n), dtype=torch.uint8, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    names = ("quench", "npe", "profile", "scintillation", "fluctuate", "electronics")
    launches0 = lartpc.kernel_launches()

    def staged():
        e = [torch.cuda.Event(enable_timing=True) for _ in range(7)]
        e[0].record(); _, ne = sim.quench(seg)
        e[1].record(); a = light.npe(seg, ne)
        e[2].record(); ipe = light.profile(a)
        e[3].record(); isc = light.scintillation(ipe)
        e[4].record(); nobs = light.fluctuate(isc, wl.seed)
        e[5].record(); v = light.electronics(nobs, wl.seed)
        e[6].record()
        torch.cuda.synchronize()
        return [e[k].elapsed_time(e[k + 1]) for k in range(6)], ipe

    for _ in range(args.warmup):
        flush.zero_(); staged()
    clocks = ClockSampler(0)
    clocks.start()
    per, steps = [], []
    for _ in range(args.steps):
        flush.zero_()
        t, ipe = staged()
        per.append(t)
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        _, ne = sim.quench(seg)
        v = light.run(seg, ne, wl.seed, workspace=ws)
        e1.record()
        torch.cuda.synchronize()
        steps.append(e0.elapsed_time(e1))
    clk = clocks.stop()
    # end to end: pinned host segments in, pinned host waveforms out
    dseg = {k: torch.empty_like(v_) for k, v_ in seg.items()}
    hv = torch.empty((n_det, int(lp["n_ticks"])), dtype=torch.float32).pin_memory()

    def e2e_step():
        for k, v_ in host.items():
            dseg[k].copy_(v_, non_blocking=True)
        _, ne_ = sim.quench(dseg)
        hv.copy_(light.run(dseg, ne_, wl.seed, workspace=ws), non_blocking=True)
        torch.cuda.synchronize()

    e2e_step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()
    e2e_ms = (time.perf_counter() - t0) * 1e3 / args.steps
    mp = {}
    try:
        mp = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm = float(mp.get("hbm_gbs", 6650.0))
    fp32 = lartpc.measure_fp32_peak(0)
    med = {k: float(np.median([p_[i] for p_ in per])) for i, k in enumerate(names)}
    ms = float(np.median(steps))
    n_t, n_sc, n_rs, n_lt = int(lp["n_ticks"]), int(lp["trunc_tau"] * lp["tau_slow_us"] / lp["tick_us"]) + 1, int(lp["n_resp"]), int(lp["n_lut_t"])
    npe_bytes = n * (36.0 + 4.0 + 12.0 + 4.0 * n_det)
    prof_bytes = n * (8.0 + n_det * (4.0 + 4.0 * n_lt))                # ids / voxels once, per sensor N_pe and one LUT profile (L2 gathers)
    rooflines = [
        {"kernel": "light_npe_kernel (L1)", "bound": "hbm", "ms_per_step": med["npe"], "moved_bytes_per_step": npe_bytes,
         "achieved": npe_bytes / (med["npe"] * 1e-3) / 1e9, "peak": hbm, "unit": "GB/s", "frac": npe_bytes / (med["npe"] * 1e-3) / 1e9 / hbm},
        {"kernel": "tick sort + light_tick_sum_kernel + light_profile_kernel (L2)", "bound": "hbm", "ms_per_step": med["profile"],
         "moved_bytes_per_step": prof_bytes, "achieved": prof_bytes / (med["profile"] * 1e-3) / 1e9, "peak": hbm, "unit": "GB/s",
         "frac": prof_bytes / (med["profile"] * 1e-3) / 1e9 / hbm,
         "note": "bytes the sums read: N_pe once per sensor, one LUT time profile per (sensor, segment) through L2"},
        {"kernel": "light_conv_kernel, scintillation (L3)", "bound": "alu", "ms_per_step": med["scintillation"],
         "achieved": 2.0 * n_det * n_t * n_sc / (med["scintillation"] * 1e-3) / 1e12, "peak": fp32, "unit": "TFLOP/s",
         "frac": 2.0 * n_det * n_t * n_sc / (med["scintillation"] * 1e-3) / 1e12 / fp32},
        {"kernel": "light_conv_kernel, read-out (L5)", "bound": "alu", "ms_per_step": med["electronics"],
         "achieved": 2.0 * n_det * n_t * n_rs / (med["electronics"] * 1e-3) / 1e12, "peak": fp32, "unit": "TFLOP/s",
         "frac": 2.0 * n_det * n_t * n_rs / (med["electronics"] * 1e-3) / 1e12 / fp32},
    ]
    print(json.dumps({
        "metric": "segments/s through the light simulation (S1 + eqs. 4.1-4.6; ms per spill in ms_per_step)", "value": n / (ms * 1e-3),
        "unit": "segments/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32 (float64 where an integer is decided)", "data": "synthetic",
        "config": {"workload": WORKLOAD_NAMES[args.config] + "; light: %d photosensors, %d ticks of %g ns, synthetic light LUT of "
                   "%d voxels x %d time bins" % (n_det, n_t, 1e3 * lp["tick_us"], ls.vis[0].size, n_lt),
                   "n_segments": n, "l2": "256 MiB flush write between timed steps"},
        "stage_ms_per_step": med, "rooflines": rooflines,
        "e2e": {"value": n / (e2e_ms * 1e-3), "unit": "segments/s", "ms_per_step": e2e_ms, "h2d_bytes_per_step": 36 * n,
                "d2h_bytes_per_step": 4 * n_det * n_t},
        "photoelectrons": float(ipe.sum().item()), "clocks": clk, "gpu_launches": int(lartpc.kernel_launches() - launches0)}))


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.light:
        run_light(args)
    elif args.config == 4:
        run_sweep(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
