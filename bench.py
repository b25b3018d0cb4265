#!/usr/bin/env python
"""bench.py -- walker local energies/s of the LO-AFQMC hot path (BASELINE.json:metric) on B200.

  python bench.py --gpus N --steps K --warmup W            # this repo's CUDA path (one rank per GPU under torchrun)
  python bench.py --impl reference --gpus N --steps K ...  # the CPU oracle, as it stands, on the box's host cores

A "step" is one pass of the whole hot path (S1 Theta, S2 one-body, S3 Coulomb, S4 exchange, S5 combine)
over one batch of N_w synthetic walkers of BASELINE.json:configs[2] (pentacene-sized; the headline config).  Setup
(lo_setup: half-rotation, pair SVDs, truncation, packing) is outside the timed region, as the paper's is.
Prints ONE JSON line on rank 0.
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

METRIC = "walker local energies/s (complex128 LO-AFQMC E_L)"
UNIT = "energies/s"
NOMINAL_FP64_TFLOPS = 40.0     # B200 datasheet FP64 (vector = tensor); context for the ratio-derived peak
NOMINAL_BF16_TFLOPS = 2250.0
# roofline.traffic = dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel, read from the
# sidecar of the committed `ncu --set full` capture (one row per workload: the two counters, the commit and the SHA-256 of
# the kernel sources the capture was taken at).  A row whose hash is not that of the kernel sources being run is stale:
# traffic is then null and `traffic_note` says why.
TRAFFIC_SIDECAR = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
KERNEL_SOURCES = ("lo_kernels.cu", "lo_device.cuh")
KERNEL_SOURCES_I8 = ("lo_exchange_i8.cu", "lo_device.cuh")     # rows whose kernel is k_exchange_i8
NOMINAL_INT8_OVER_BF16 = 2.0   # dense INT8 : bf16 tensor throughput (4.5 : 2.25 POP/s), B200_PROFILING.md nominal table (fp8 row; kind::i8 runs at the fp8 rate)


def kernel_sources_sha256(names=KERNEL_SOURCES):
    import hashlib
    h = hashlib.sha256()
    for name in names:
        with open(os.path.join(ROOT, "paper_2202_00832_b200", "csrc", name), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def ncu_traffic(workload, int8=False):
    """(bytes per launch or None, note) for `workload` from profiles/ncu_traffic.csv; int8: the row of k_exchange_i8."""
    import csv
    names = KERNEL_SOURCES_I8 if int8 else KERNEL_SOURCES
    try:
        with open(TRAFFIC_SIDECAR, newline="") as fh:
            rows = [r for r in csv.DictReader(fh) if r["workload"] == workload and r["kernel"].startswith("k_exchange_i8") == int8]
    except OSError:
        return None, "no sidecar %s" % os.path.relpath(TRAFFIC_SIDECAR, ROOT)
    if not rows:
        return None, "no ncu --set full capture of this workload in %s" % os.path.relpath(TRAFFIC_SIDECAR, ROOT)
    sha = kernel_sources_sha256(names)
    fresh = [r for r in rows if r["kernel_sources_sha256"] == sha]
    if not fresh:
        return None, "capture of commit %s is stale: %s changed since (sha256 %s.. != %s..)" % (
            rows[-1]["commit"], "+".join(names), rows[-1]["kernel_sources_sha256"][:12], sha[:12])
    r = fresh[-1]
    return float(r["dram_bytes_read"]) + float(r["dram_bytes_write"]), "%s of %s at commit %s (%s)" % (
        r["kernel"], r["capture"], r["commit"], "dram__bytes_read.sum + dram__bytes_write.sum")


def workload_name(cfg, reading, T, n_w):
    import gen
    spec = gen.CONFIGS[cfg]
    return "configs[%d] %s, %s reading, T_SVD=%g, N_w=%d" % (cfg, spec.name, reading, T, n_w)


class ClockSampler:
    """nvidia-smi sampled every 100 ms while the timed region runs (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc, self.th = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.th = threading.Thread(target=self._read, daemon=True)
        self.th.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        rows = [r for t, r in self.rows if t0 <= t <= t1 and len(r) >= 7] or [r for _, r in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[3 + k].lower().startswith("active") for r in rows)]
        pw = [float(r[2]) for r in rows if r[2].replace(".", "", 1).isdigit()]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "reasons": reasons, "samples": len(rows),
                "power_w_max": max(pw) if pw else None}


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


def oracle_inputs_from_library(P, F):
    """Host copies the oracle needs to evaluate on the LIBRARY's factor set (parity protocol A)."""
    import oracle
    hr = [oracle.half_rotate(P.L, P.h, psi) for psi in P.psi]
    fs = []
    for s in range(P.n_spin):
        U, sg, W = F.factor_all(s)
        pi, pj = oracle.all_pairs(P.n_occ[s])
        fs.append(oracle.make_factor_set(P.N, P.n_occ[s], pi, pj, F.ranks(s), U, sg, W))
    return [a for a, _ in hr], [b for _, b in hr], fs


def run_ours(args):
    import torch
    import torch.distributed as dist

    import gen
    import paper_2202_00832_b200 as lo
    from paper_2202_00832_b200.dist import max_over_ranks

    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    cfg, reading = args.config, args.reading
    spec = gen.CONFIGS[cfg]
    T = args.threshold if args.threshold is not None else spec.thresholds[0]
    n_w = args.walkers or spec.n_w

    t0 = time.time()
    P = gen.make_problem(cfg, reading=reading)          # same seed on every rank: the factor set is replicated
    F = lo.Factors.setup(P.h, P.L, P.psi, T, device=local, max_walkers=n_w, gpu_svd=True, propagator=args.propagator)
    info = F.info()
    setup_s = time.time() - t0
    # weak scaling: every rank owns a full batch of n_w walkers (its own seed); no data-path collective
    phis = gen.make_walkers(P, n_w, seed=P.seed + 1000 * rank)
    dphi = [torch.from_numpy(p).to(dev) for p in phis]
    fl = F.flops_per_walker()
    flops_walker = sum(v for k, v in fl.items() if k != "propagator")     # the steps of lo_local_energy (S1-S5)

    peak_dmma = lo.measure_peak("dmma", local)
    peak_dfma = lo.measure_peak("dfma", local)
    peak_hbm = lo.measure_peak("hbm", local)

    # ---- exchange route of the timed step.  "int8" (default): projections from exact INT8 digit slices on the tcgen05 tensor cores
    # and the Coulomb / one-body contraction on the same route (lo_set_exchange_mode, parity-tested at the same 1e-10); the FP64 DMMA
    # route of the same factor set is timed first, with the
    # same warm-up and step count, and reported as `dmma_route` (its own roofline against the measured FP64 peak).
    int8 = args.exchange == "int8"
    dmma_route = None
    if int8:
        for _ in range(max(args.warmup, 3)):
            F.local_energy(dphi, parts=True)
        torch.cuda.synchronize()
        F.timing_enable(True)
        F.timing_get()
        d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        d0.record()
        for _ in range(args.steps):
            out_d = F.local_energy(dphi, parts=True)
        d1.record()
        torch.cuda.synchronize()
        tmd = F.timing_get()
        F.timing_enable(False)
        d_ms = max_over_ranks(d0.elapsed_time(d1), dev)
        dx_ms = tmd["exchange"][0] / max(tmd["exchange"][1], 1)
        dx_tf = fl["exchange"] * n_w / (dx_ms * 1e-3) * 1e-12
        E_dmma = torch.stack(out_d[:4], dim=1).cpu().numpy()
        tr_d, tr_d_note = ncu_traffic(workload_name(cfg, reading, T, n_w))
        dmma_route = {"what": "same step with lo_set_exchange_mode(LO_EXCHANGE_DMMA): k_exchange on the FP64 tensor pipe",
                      "value": round(world * n_w * args.steps / (d_ms * 1e-3), 2), "unit": UNIT, "ms_per_step": round(d_ms / args.steps, 4),
                      "roofline": {"bound": "tensor", "kernel": "k_exchange (grouped variable-rank dual DGEMM + fused sigma-weighted a.b)",
                                   "achieved": round(dx_tf, 3), "peak": round(max(peak_dmma, peak_dfma), 3), "unit": "TFLOP/s",
                                   "frac": round(dx_tf / max(peak_dmma, peak_dfma), 4), "kernel_ms": round(dx_ms, 4),
                                   "traffic": tr_d, "traffic_note": tr_d_note}}
        F.set_exchange_mode(True)
    for _ in range(max(args.warmup, 3)):
        F.local_energy(dphi, parts=True)
    torch.cuda.synchronize()
    F.timing_enable(True)
    F.timing_get()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    tw0 = time.time()
    ev0.record()
    for _ in range(args.steps):
        out = F.local_energy(dphi, parts=True)
    ev1.record()
    torch.cuda.synchronize()
    tw1 = time.time()
    if world > 1:
        dist.barrier()
    ms = ev0.elapsed_time(ev1)
    clocks = sampler.stop(tw0, tw1)
    ms_max = max_over_ranks(ms, dev)
    tm = F.timing_get()
    F.timing_enable(False)
    n_kernels = sum(n for _, n in tm.values()) + tm["coulomb"][1]      # the coulomb bracket holds 2 launches (GEMM + k_ej)
    if int8:
        n_kernels += tm["coulomb"][1] + tm["exchange"][1]              # + k_slice_theta (coulomb bracket), + k_i8_poison (exchange bracket)
    value = world * n_w * args.steps / (ms_max * 1e-3)

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D of Phi and D2H of E inside the timed region
    pinned = [torch.from_numpy(p).pin_memory() for p in phis]
    E_host = torch.empty((n_w, 4), dtype=torch.complex128).pin_memory()
    st_host = torch.empty(n_w, dtype=torch.int32).pin_memory()
    for _ in range(2):
        F.local_energy_host(pinned, E_host, st_host)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        F.local_energy_host(pinned, E_host, st_host)
    e1.record()
    torch.cuda.synchronize()
    ms_e2e = max_over_ranks(e0.elapsed_time(e1), dev)
    h2d = sum(p.numel() * 16 for p in pinned)
    d2h = n_w * 4 * 16 + n_w * 4
    e2e_value = world * n_w * args.steps / (ms_e2e * 1e-3)
    E_dev = torch.stack(out[:4], dim=1).cpu().numpy()
    # the host variant runs the batch in walker chunks (H2D of chunk c+1 under the kernels of chunk c): same arithmetic,
    # another fixed summation order of the per-CTA partials
    assert (np.abs(E_host.numpy() - E_dev).max(axis=1) <= 1e-12 * np.abs(E_dev[:, 0])).all(), "host-buffer path and device path disagree"

    # ---- roofline of the dominant kernel (exchange grouped GEMM), timed live with CUDA events on the launch stream
    ex_ms, ex_n = tm["exchange"]
    ex_avg = ex_ms / max(ex_n, 1)
    ex_flops = fl["exchange"] * n_w
    achieved = ex_flops / (ex_avg * 1e-3) * 1e-12
    peak = max(peak_dmma, peak_dfma)
    mp = measured_peaks()
    if not int8:
        traffic, traffic_note = ncu_traffic(workload_name(cfg, reading, T, n_w))
        roofline = {"bound": "tensor", "kernel": "k_exchange (grouped variable-rank dual DGEMM + fused sigma-weighted a.b)",
                    "achieved": round(achieved, 3), "peak": round(peak, 3), "unit": "TFLOP/s", "frac": round(achieved / peak, 4),
                    "traffic": traffic, "traffic_note": traffic_note,
                    "peak_source": "in-run register-resident DMMA.8x8x4 / DFMA loops (lo_measure_peak), of measured",
                    "peak_dmma": round(peak_dmma, 3), "peak_dfma": round(peak_dfma, 3),
                    "peak_from_bf16_ratio": round(mp.get("bf16_tflops", 0) * NOMINAL_FP64_TFLOPS / NOMINAL_BF16_TFLOPS, 2) if mp else None,
                    "hbm_gbs_in_run": round(peak_hbm, 1), "hbm_gbs_measured_peaks": mp.get("hbm_gbs"),
                    "kernel_ms": round(ex_avg, 4), "kernel_share_of_step": round(ex_ms / max(sum(m for m, _ in tm.values()), 1e-9), 4),
                    "algorithmic_flops_per_launch": ex_flops,
                    "algorithmic_bytes_per_launch": 16.0 * info.N * sum(info.sum_rank) + 8.0 * sum(info.sum_rank) + 16.0 * info.N * sum(info.n_occ) * n_w}
    else:
        # k_exchange_i8: every fp64 multiply-add of the two projections becomes 28 INT8 multiply-adds (7 x 7 digits, index sum <= 6)
        # on the tcgen05 tensor cores.  achieved = those algorithmic integer ops / the exchange bracket (k_exchange_i8 + the
        # one-block k_i8_poison; the per-call slicing of Theta, k_slice_theta, sits in the coulomb bracket, whose INT8 GEMM
        # k_coulomb_i8 uses the digits first); peak = measured dense bf16 (MEASURED_PEAKS.json, burst) x the nominal
        # INT8 : bf16 ratio of 2, else the guide's nominal fallback.
        r_sum = float(sum(info.sum_rank))
        i8_ops = 28.0 * 8.0 * info.N * r_sum * n_w
        achieved_i8 = i8_ops / (ex_avg * 1e-3) * 1e-12
        bf16 = mp.get("bf16_tflops")
        peak_i8 = (bf16 if bf16 else NOMINAL_BF16_TFLOPS) * NOMINAL_INT8_OVER_BF16
        traffic, traffic_note = ncu_traffic(workload_name(cfg, reading, T, n_w), int8=True)
        roofline = {"bound": "tensor", "kernel": "k_exchange_i8 (grouped dual GEMM from 7 x 7 INT8 digit slices, tcgen05.mma kind::i8 into TMEM, fused fp64 "
                                                 "recombination + sigma-weighted a.b)",
                    "achieved": round(achieved_i8, 1), "peak": round(peak_i8, 1), "unit": "TFLOP/s", "frac": round(achieved_i8 / peak_i8, 4),
                    "unit_note": "integer ops (2 per INT8 multiply-add) of the 28 digit products per fp64 multiply-add",
                    "traffic": traffic, "traffic_note": traffic_note,
                    "peak_source": ("MEASURED_PEAKS.json bf16_tflops (burst) x 2 (nominal INT8 : bf16)" if bf16 else
                                    "fallback: nominal dense bf16 2250 TFLOP/s x 2 (B200_PROFILING.md); MEASURED_PEAKS.json absent"),
                    "peak_bf16_sustained_x2": round(mp["bf16_tflops_sustained"] * NOMINAL_INT8_OVER_BF16, 1) if mp.get("bf16_tflops_sustained") else None,
                    "fp64_equivalent_tflops": round(achieved, 3), "fp64_equivalent_over_measured_dmma_peak": round(achieved / peak, 4),
                    "peak_dmma": round(peak_dmma, 3), "peak_dfma": round(peak_dfma, 3),
                    "hbm_gbs_in_run": round(peak_hbm, 1), "hbm_gbs_measured_peaks": mp.get("hbm_gbs"),
                    "kernel_ms": round(ex_avg, 4), "kernel_share_of_step": round(ex_ms / max(sum(m for m, _ in tm.values()), 1e-9), 4),
                    "algorithmic_int8_ops_per_launch": i8_ops, "algorithmic_flops_per_launch_fp64": ex_flops,
                    "algorithmic_bytes_per_launch": 14.0 * info.N * r_sum + 8.0 * r_sum + 14.0 * info.N * sum(info.n_occ) * n_w,
                    "int8_slices_GB": round(F.info().int8_bytes / 1e9, 3)}
        dmma_route["max_rel_diff_int8_vs_dmma"] = float((np.abs(E_dev - E_dmma).max(axis=1) / np.abs(E_dmma[:, 0])).max())
    # per STEP (an unrestricted config launches the S1 kernels once per spin; flops_per_walker sums both spins)
    kernels = {k: {"ms": round(m / args.steps, 4), "tflops": round(fl[k] * n_w / (m / args.steps * 1e-3) * 1e-12, 3) if m > 0 else 0.0}
               for k, (m, n) in tm.items()}

    # ---- SURVEY 8(f) NEXT-1 (outside the timed step and outside `value`): propagator formation B_w = sum_g x^g_w L^g
    nxt = None
    if args.propagator:
        gx = torch.Generator(device=dev).manual_seed(P.seed + rank)
        x = torch.randn((n_w, info.n_chol, 2), dtype=torch.float64, device=dev, generator=gx)
        x = torch.view_as_complex(x).contiguous()
        def time_propagator():
            for _ in range(3):
                F.propagator(x)
            torch.cuda.synchronize()
            F.timing_enable(True)
            F.timing_get()
            for _ in range(args.steps):
                F.propagator(x)
            torch.cuda.synchronize()
            pm, pn = F.timing_get()["propagator"]
            F.timing_enable(False)
            return pm / max(pn, 1)
        p_ms = time_propagator()
        p_tf = fl["propagator"] * n_w / (p_ms * 1e-3) * 1e-12
        if int8:
            # fp64-equivalent rate of the INT8 route (28 digit products per multiply-add), next to the DMMA route of the same call
            F.set_exchange_mode(False)
            pd_ms = time_propagator()
            F.set_exchange_mode(True)
            pd_tf = fl["propagator"] * n_w / (pd_ms * 1e-3) * 1e-12
            nxt = {"propagator": {"what": "B_w = sum_g x^g_w L^g for all walkers, upper triangle (PAPER.md:310): k_pack_x + k_slice_theta + k_coulomb_i8 "
                                          "(INT8 digit slices on tcgen05)",
                                  "ms": round(p_ms, 4), "fp64_equivalent_tflops": round(p_tf, 3), "fp64_equivalent_over_measured_dmma_peak": round(p_tf / peak, 4),
                                  "dmma_route_ms": round(pd_ms, 4), "dmma_route_tflops": round(pd_tf, 3), "dmma_route_frac_of_peak": round(pd_tf / peak, 4),
                                  "flops_per_walker": fl["propagator"]}}
        else:
            nxt = {"propagator": {"what": "B_w = sum_g x^g_w L^g for all walkers, upper triangle (PAPER.md:310), k_pack_x + DMMA GEMM",
                                  "ms": round(p_ms, 4), "tflops": round(p_tf, 3), "frac_of_peak": round(p_tf / peak, 4),
                                  "flops_per_walker": fl["propagator"]}}

    # ---- SURVEY 8(f) NEXT-3 (outside `value`): the paper-literal energy, Coulomb term from the compressed factors too
    if info.n_spin == 1:
        F.set_coulomb_mode(True)        # in the mode of the timed step: four projections per pair from the INT8 digits, or DMMA
        flc = F.flops_per_walker()
        for _ in range(3):
            F.local_energy(dphi, parts=True)
        torch.cuda.synchronize()
        F.timing_enable(True)
        F.timing_get()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record()
        for _ in range(args.steps):
            F.local_energy(dphi, parts=True)
        c1.record()
        torch.cuda.synchronize()
        cm, cn = F.timing_get()["exchange"]
        F.timing_enable(False)
        F.set_coulomb_mode(False)
        c_ms = cm / max(cn, 1)
        c_tf = flc["exchange"] * n_w / (c_ms * 1e-3) * 1e-12
        nxt = dict(nxt or {})
        nxt["compressed_coulomb"] = {"what": "lo_set_coulomb_mode(COMPRESSED): E_J and E_K both from the pair factors (Eq. 19/22), 4 projections per pair"
                                             + (" on the INT8 route (exchange_tflops is fp64-equivalent)" if int8 else ""),
                                     "ms_per_step": round(c0.elapsed_time(c1) / args.steps, 4),
                                     "energies_per_s": round(n_w * args.steps / (c0.elapsed_time(c1) * 1e-3), 2),
                                     "exchange_ms": round(c_ms, 4), "exchange_tflops": round(c_tf, 3), "exchange_frac_of_peak": round(c_tf / peak, 4)}

    # ---- gated experiment (never part of `value` or of the product path): one FP64-accurate GEMM tile from INT8 slices
    # on tcgen05, against the same tile's cost at the measured DMMA peak
    if rank == 0:
        try:
            p_us, p_err = lo.measure_peak("int8_tile_us", local), lo.measure_peak("int8_tile_err", local)
            dmma_us = 2.0 * 128 * 128 * 384 / (peak_dmma * 1e12 / torch.cuda.get_device_properties(local).multi_processor_count) * 1e6
            nxt = dict(nxt or {})
            nxt["int8_slicing_probe"] = {"what": "128 x 128 x 384 fp64 tile from 6 x 6 INT8 slices (21 digit products, tcgen05.mma kind::i8, TMEM, fp64 "
                                                 "recombination); operands resident in shared memory: the operand feed is not measured",
                                         "us_per_tile": round(p_us, 3), "max_err_vs_fp64_rel_to_max": p_err,
                                         "same_tile_at_measured_dmma_peak_us": round(dmma_us, 3), "ratio": round(dmma_us / p_us, 2)}
        except lo.LoError as e:
            nxt = dict(nxt or {})
            nxt["int8_slicing_probe"] = {"error": str(e)}

    # ---- SURVEY 8(f) NEXT-2 (opt-in, outside `value`): multi-determinant trial by direct summation, own factor set
    if args.cas > 0 and info.n_spin == 1:
        n_virt, n_real = 6, max(1, n_w // args.cas)
        Tr = gen.make_cas_trial(P, n_virt=n_virt, n_act_occ=6, n_det=args.cas, max_exc=4)
        Fc = lo.Factors.setup(P.h, P.L, [Tr.C], T, device=local, max_walkers=n_real * args.cas, gpu_svd=True)
        Fc.set_cas_trial(Tr.n_ref, Tr.holes, Tr.parts, Tr.coef, n_real)
        phic = dphi[0][:n_real].contiguous()
        for _ in range(3):
            Fc.local_energy_cas(phic)
        torch.cuda.synchronize()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record()
        for _ in range(args.steps):
            Fc.local_energy_cas(phic)
        c1.record()
        torch.cuda.synchronize()
        cas_ms = c0.elapsed_time(c1) / args.steps
        nxt = dict(nxt or {})
        nxt["cas_trial_direct"] = {"what": "lo_local_energy_cas, LO_CAS_DIRECT: %d determinants (<= 4 excitations, 6 active occupied x %d virtuals), %d real "
                                           "walkers = %d virtual walkers, SMW Green's functions + the ordinary kernels" % (args.cas, n_virt, n_real, n_real * args.cas),
                                   "ms_per_step": round(cas_ms, 4), "energies_per_s": round(n_real / (cas_ms * 1e-3), 2),
                                   "determinant_energies_per_s": round(n_real * args.cas / (cas_ms * 1e-3), 2)}
        # the rearranged SMW energy (Eq. 21-23) on the same trial and factor set, all real walkers the workspace allows
        n_smw = min(n_w, n_real * args.cas)
        Fc.set_cas_trial(Tr.n_ref, Tr.holes, Tr.parts, Tr.coef, n_smw, smw_energy=True)
        phism = dphi[0][:n_smw].contiguous()
        for _ in range(3):
            Fc.local_energy_cas(phism)
        torch.cuda.synchronize()
        c0.record()
        for _ in range(args.steps):
            Fc.local_energy_cas(phism)
        c1.record()
        torch.cuda.synchronize()
        smw_ms = c0.elapsed_time(c1) / args.steps
        nxt["cas_trial_smw"] = {"what": "lo_local_energy_cas, LO_CAS_SMW_ENERGY (Eq. 21-23): same %d determinants, %d real walkers" % (args.cas, n_smw),
                                "ms_per_step": round(smw_ms, 4), "energies_per_s": round(n_smw / (smw_ms * 1e-3), 2),
                                "determinant_energies_per_s": round(n_smw * args.cas / (smw_ms * 1e-3), 2),
                                "speedup_vs_direct_per_walker": round((cas_ms / n_real) / (smw_ms / n_smw), 2)}
        Fc.free()

    cpu_baseline = None
    if rank == 0 and world == 1 and args.cpu_walkers > 0:
        import oracle
        Lbars, hbars, fs = oracle_inputs_from_library(P, F)
        nb = min(args.cpu_walkers, n_w)
        sel = [p[:nb] for p in phis]
        t = time.time()
        Eo, _ = oracle.local_energy_lo(P.psi, Lbars, hbars, fs, sel)
        dt = time.time() - t
        err = float((np.abs(E_dev[:nb] - Eo) / np.abs(Eo[:, :1])).max())
        cpu_baseline = {"value": round(nb / dt, 3), "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                        "sample": "first %d of %d walkers of the same batch, library factor set, %.1f s" % (nb, n_w, dt),
                        "max_rel_err_gpu_vs_oracle": err}

    if rank == 0:
        line = {"metric": METRIC, "value": round(value, 2), "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
                "ms_per_step": round(ms_max / args.steps, 4), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "s8 x s8 -> s32 digit products + f64 recombination (exchange, Coulomb), f64 (everything else)" if int8 else "f64",
                "data": "synthetic",
                "config": {"workload": workload_name(cfg, reading, T, n_w), "N": info.N, "N_occ": list(info.n_occ)[:info.n_spin],
                           "N_chol": info.n_chol, "N_w_per_gpu": n_w, "T_SVD": T, "sum_rank": sum(info.sum_rank),
                           "compression_pct": round(100 * (1 - sum(info.sum_rank) / (sum(info.n_pairs) * info.N)), 2),
                           "factor_GB": round(info.factor_bytes / 1e9, 3), "parallelism": "walker-sharded replicas x%d, no collective" % world,
                           "l2": "inputs larger than L2 (factor set %.1f GB, Theta %.0f MB per step)" % (
                               info.factor_bytes / 1e9, 16e-6 * info.N_pad * sum(info.n_occ) * n_w),
                           "setup_s": round(setup_s, 1), "lo_setup_s": round(info.setup_seconds, 2), "setup_svd_s": round(info.setup_svd_seconds, 2),
                           "svd_sweeps_max": info.svd_sweeps_max, "pairs_prescreened": int(info.n_pairs_prescreened)},
                "tflops": round(flops_walker * n_w * world * args.steps / (ms_max * 1e-3) * 1e-12, 3),
                "tflops_note": "algorithmic complex128 flops of S1-S5 per second (fp64-equivalent when the exchange runs from INT8 slices)",
                "flops_per_walker": flops_walker, "kernels": kernels, "roofline": roofline, "cpu_baseline": cpu_baseline,
                "e2e": {"value": round(e2e_value, 2), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                        "ms_per_step": round(ms_e2e / args.steps, 4), "api": "lo_local_energy_host (C ABI, pinned host buffers)"},
                "gpu_launches": int(n_kernels), "clocks": clocks, "exchange": args.exchange,
                "precision_note": ("fp64-accurate result, not a reduced-precision one: the INT8 route multiplies EXACT 7-bit integer digits of the fp64 operands "
                                   "(28 digit products per multiply-add, exact in int32) and recombines in fp64; parity bar 1e-10 of |E_L| per walker "
                                   "(tests/test_gpu_parity.py), measured in this run: %.1e against the DMMA route over all walkers%s" % (
                                       dmma_route["max_rel_diff_int8_vs_dmma"],
                                       ", %.1e against the CPU oracle on the sampled walkers" % cpu_baseline["max_rel_err_gpu_vs_oracle"] if cpu_baseline else ""))
                if int8 else "fp64 throughout (DMMA tensor pipe)",
                "dmma_route": dmma_route, "next": nxt}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_sweep(args):
    """BASELINE.json:configs[4] threshold sweep: the factor set is built ONCE at the tightest threshold (device SVD) and
    re-truncated (prefix truncation, lo_retruncate) to each looser one; per threshold one JSON line with sum r_ij,
    factor bytes, compression, E_K error against the exact full-ERI/Cholesky exchange (oracle, a few walkers), the
    truncation bound (R5) and throughput.  Not the default bench line; one GPU."""
    import concurrent.futures as cf

    import torch

    import gen
    import oracle
    import paper_2202_00832_b200 as lo
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(0)
    cfg, reading = args.config, args.reading
    spec = gen.CONFIGS[cfg]
    Ts = sorted(spec.thresholds if args.threshold is None else [args.threshold])
    n_w = args.walkers or spec.n_w
    P = gen.make_problem(cfg, reading=reading)
    phis = gen.make_walkers(P, n_w)
    dphi = [torch.from_numpy(p).cuda() for p in phis]
    t0 = time.time()
    F0 = lo.Factors.setup(P.h, P.L, P.psi, Ts[0], device=0, max_walkers=n_w, gpu_svd=True)
    setup_s = time.time() - t0
    peak = max(lo.measure_peak("dmma", 0), lo.measure_peak("dfma", 0))
    # exact exchange (Eq. 16, oracle O2) and the norms of the R5 bound for a few seeded walkers
    idx = np.sort(np.random.default_rng(P.seed).choice(n_w, min(args.sweep_exact_walkers, n_w), replace=False))
    hr = [oracle.half_rotate(P.L, P.h, psi) for psi in P.psi]
    cK = 1.0 if P.n_spin == 1 else 0.5

    def exact_one(w):
        ek, nrm = 0.0, []
        for s in range(P.n_spin):
            th, _, _ = oracle.theta(P.psi[s], phis[s][w])
            ek += cK * oracle.exchange_cholesky(hr[s][0], th)
            nrm.append(np.linalg.norm(th, axis=0))
        return ek, nrm

    t0 = time.time()
    with cf.ThreadPoolExecutor(max_workers=max(1, len(idx))) as ex:
        exact = list(ex.map(exact_one, idx))
    exact_s = time.time() - t0
    rows = []
    for T in Ts:
        F = F0 if T == Ts[0] else F0.retruncate(T)
        info = F.info()
        fl = F.flops_per_walker()
        for _ in range(max(args.warmup, 3)):
            out = F.local_energy(dphi, parts=True)
        torch.cuda.synchronize()
        F.timing_enable(True)
        F.timing_get()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        for _ in range(args.steps):
            out = F.local_energy(dphi, parts=True)
        ev1.record()
        torch.cuda.synchronize()
        ms = ev0.elapsed_time(ev1) / args.steps
        tm = F.timing_get()
        F.timing_enable(False)
        EK = out[3].cpu().numpy()
        ex_ms = tm["exchange"][0] / max(tm["exchange"][1], 1)
        errs, bounds = [], []
        for (ek, nrm), w in zip(exact, idx):
            errs.append(abs(EK[w] - ek))
            b = 0.0
            for s in range(P.n_spin):
                pi, pj = oracle.all_pairs(P.n_occ[s])
                m = np.where(pi == pj, 1.0, 2.0)
                b += cK * T * float((m * nrm[s][pi] * nrm[s][pj]).sum())
            bounds.append(b)
        sum_r = int(sum(info.sum_rank))
        row = {"sweep": workload_name(cfg, reading, T, n_w), "T_SVD": T, "sum_rank": sum_r, "min_rank": info.min_rank,
               "max_rank": info.max_rank, "compression_pct": round(100 * (1 - sum_r / (sum(info.n_pairs) * info.N)), 2),
               "factor_bytes": int(info.factor_bytes), "EK_abs_err_vs_exact_max": float(max(errs)),
               "EK_abs_err_vs_exact_mean": float(np.mean(errs)), "EK_exact_abs_mean": float(np.mean([abs(e) for e, _ in exact])),
               "R5_bound_min": float(min(bounds)), "exact_walkers": [int(w) for w in idx],
               "ms_per_step": round(ms, 3), "energies_per_s": round(n_w / (ms * 1e-3), 2),
               "tflops": round(sum(v for k, v in fl.items() if k != "propagator") * n_w / (ms * 1e-3) * 1e-12, 3), "exchange_ms": round(ex_ms, 3),
               "exchange_tflops": round(fl["exchange"] * n_w / (ex_ms * 1e-3) * 1e-12, 3) if ex_ms > 0 else 0.0,
               "exchange_frac_of_peak": round(fl["exchange"] * n_w / (ex_ms * 1e-3) * 1e-12 / peak, 4) if ex_ms > 0 else 0.0,
               "peak_tflops": round(peak, 3), "setup_s_tightest": round(setup_s, 1), "oracle_exact_s": round(exact_s, 1)}
        # ---- the same factor set on the INT8 route (exchange + Coulomb from digit slices on tcgen05), when its digits fit beside
        # what is resident (the sweep keeps the tightest set alive for the re-truncations: run one threshold per invocation,
        # --threshold T, to get this leg at every threshold of configs[4])
        if args.exchange == "int8":
            need = 0.9 * info.factor_bytes + 1.0 * info.lbar_bytes + (2 << 30)
            free_b = torch.cuda.mem_get_info()[0]
            if free_b < need:
                row["int8"] = {"skipped": "digits need %.1f GB, %.1f GB free" % (need / 1e9, free_b / 1e9)}
            else:
                E_d = torch.stack(out[:4], dim=1).cpu().numpy()
                F.set_exchange_mode(True)
                for _ in range(max(args.warmup, 3)):
                    out = F.local_energy(dphi, parts=True)
                torch.cuda.synchronize()
                F.timing_enable(True)
                F.timing_get()
                ev0.record()
                for _ in range(args.steps):
                    out = F.local_energy(dphi, parts=True)
                ev1.record()
                torch.cuda.synchronize()
                ms8 = ev0.elapsed_time(ev1) / args.steps
                tm8 = F.timing_get()
                F.timing_enable(False)
                F.set_exchange_mode(False)
                E_q = torch.stack(out[:4], dim=1).cpu().numpy()
                ex8 = tm8["exchange"][0] / max(tm8["exchange"][1], 1)
                EK8 = E_q[:, 3]
                row["int8"] = {"ms_per_step": round(ms8, 3), "energies_per_s": round(n_w / (ms8 * 1e-3), 2), "exchange_ms": round(ex8, 3),
                               "coulomb_ms": round(tm8["coulomb"][0] / max(tm8["coulomb"][1], 1), 3),
                               "exchange_fp64_equivalent_tflops": round(fl["exchange"] * n_w / (ex8 * 1e-3) * 1e-12, 2),
                               "exchange_int8_pops": round(28.0 * 8.0 * info.N * sum_r * n_w / (ex8 * 1e-3) * 1e-15, 3),
                               "max_rel_diff_vs_dmma_route": float((np.abs(E_q - E_d).max(axis=1) / np.abs(E_d[:, 0])).max()),
                               "EK_abs_err_vs_exact_max": float(max(abs(EK8[w] - ek) for (ek, _), w in zip(exact, idx))),
                               "int8_slices_GB": round(F.info().int8_bytes / 1e9, 2)}
        print(json.dumps(row), flush=True)
        rows.append(row)
        if F is not F0:
            F.free()
    F0.free()


def run_screen(args):
    """--screen: the pair-screening study ("reduce the number of pairs to N from N^2") on
    chains of growing length (3 functions and one occupied orbital per site, N_chol = 5N, T_SVD = 1e-5, spacing 1.4): per
    chain the pairs removed by the rigorous pre-SVD screen, and per energy-screen cutoff the kept pairs, sum r_ij, the
    largest |dE_K| over the batch against the unscreened GPU result with its bound, the error against the exact
    (Cholesky-route, oracle) exchange of two walkers, and the throughput.  One JSON line per (chain, cutoff); one GPU."""
    import torch

    import gen
    import oracle
    import paper_2202_00832_b200 as lo
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(0)
    n_w, T = args.walkers or 256, args.threshold if args.threshold is not None else 1e-5
    for n_sites in args.screen_sites:
        xyz, fns = gen.chain_geometry(n_sites, 3)
        P = gen.make_problem_from_geometry(xyz, fns, (n_sites,), 15 * n_sites, seed=3, name="chain%d" % n_sites)
        F0 = lo.Factors.setup(P.h, P.L, P.psi, T, device=0, max_walkers=n_w, gpu_svd=True)
        i0 = F0.info()
        phis = gen.make_walkers(P, n_w)
        dphi = [torch.from_numpy(p).cuda() for p in phis]
        E0 = torch.stack(F0.local_energy(dphi)[:4], dim=1).cpu().numpy()
        Lbar, _ = oracle.half_rotate(P.L, P.h, P.psi[0])
        exact = {}
        for w in (0, n_w // 2):
            th, _, _ = oracle.theta(P.psi[0], phis[0][w])
            exact[w] = (oracle.exchange_cholesky(Lbar, th), float(np.linalg.norm(th, axis=0).max()))
        for cutoff in args.screen_cutoffs:
            F = F0 if cutoff == 0 else F0.screen_pairs(cutoff)
            info = F.info()
            for _ in range(max(args.warmup, 3)):
                out = F.local_energy(dphi)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(args.steps):
                out = F.local_energy(dphi)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / args.steps
            EK = out[3].cpu().numpy()
            r = F.ranks()
            print(json.dumps({"screen": "chain of %d sites, N=%d, N_occ=%d, N_chol=%d, T_SVD=%g, N_w=%d" % (n_sites, P.N, n_sites, 15 * n_sites, T, n_w),
                              "pairs": int(i0.n_pairs[0]), "pairs_prescreened_no_svd": int(i0.n_pairs_prescreened),
                              "pair_cutoff": cutoff, "pairs_energy_screened": int(info.n_pairs_energy_screened), "pairs_kept": int((r > 0).sum()),
                              "pairs_kept_per_orbital": round(float((r > 0).sum()) / n_sites, 2), "sum_rank": int(r.sum()),
                              "dEK_vs_unscreened_max": float(np.abs(EK - E0[:, 3]).max()),
                              "dEK_bound_sum_m_sigma1": float(info.energy_screen_bound),
                              "EK_err_vs_exact": [float(abs(EK[w] - ek)) for w, (ek, _) in exact.items()],
                              "EK_exact_abs": [float(abs(ek)) for ek, _ in exact.values()],
                              "theta_norm_max": [nm for _, nm in exact.values()],
                              "ms_per_step": round(ms, 4), "energies_per_s": round(n_w / (ms * 1e-3), 1),
                              "setup_s": round(i0.setup_seconds, 2), "setup_svd_s": round(i0.setup_svd_seconds, 2)}), flush=True)
            if F is not F0:
                F.free()
        F0.free()


def run_reference(args):
    """The CPU oracle, as it stands, end to end on its OWN factors.  Its pair SVDs at the pentacene size take ~2 s per
    pair per core, so the exchange is timed on a seeded, |i-j|-stratified subset of pairs and the exchange time is
    scaled to the full pair count; Theta, one-body and Coulomb are timed in full.  A reported baseline, not a target."""
    rank = int(os.environ.get("RANK", 0))
    if rank != 0:
        return
    import gen
    import oracle
    cfg, reading = args.config, args.reading
    spec = gen.CONFIGS[cfg]
    T = args.threshold if args.threshold is not None else spec.thresholds[0]
    n_w = args.walkers or spec.n_w
    P = gen.make_problem(cfg, reading=reading)
    hr = [oracle.half_rotate(P.L, P.h, psi) for psi in P.psi]
    Lbars, hbars = [a for a, _ in hr], [b for _, b in hr]
    rng = np.random.default_rng(P.seed)
    fs, frac = [], []
    for s in range(P.n_spin):
        pi, pj = oracle.all_pairs(P.n_occ[s])
        n_sub = min(len(pi), args.ref_pairs)
        order = np.argsort(pj - pi, kind="stable")
        sub = np.sort(order[np.linspace(0, len(pi) - 1, n_sub).astype(int)]) if n_sub < len(pi) else np.arange(len(pi))
        Ut, sg, Wt = oracle.full_svd_pairs(Lbars[s], pi[sub], pj[sub])
        fs.append(oracle.truncate(P.N, P.n_occ[s], pi[sub], pj[sub], Ut, sg, Wt, T))
        frac.append(len(sub) / len(pi))
    empty = [oracle.truncate(P.N, P.n_occ[s], np.zeros(0, np.int32), np.zeros(0, np.int32), np.zeros((0, P.N, P.N)),
                             np.zeros((0, P.N)), np.zeros((0, P.N, P.N)), T) for s in range(P.n_spin)]
    nb = min(args.ref_walkers, n_w)
    phis = gen.make_walkers(P, n_w, seed=P.seed)
    sel = [p[:nb] for p in phis]
    walls, fulls = [], []
    for it in range(args.warmup + args.steps):
        t = time.time()
        oracle.local_energy_lo(P.psi, Lbars, hbars, empty, sel)
        t_base = time.time() - t
        t = time.time()
        oracle.local_energy_lo(P.psi, Lbars, hbars, fs, sel)
        t_sub = time.time() - t
        if it >= args.warmup:
            walls.append(t_base + t_sub)                                                   # what this iteration really took
            fulls.append(t_base + max(t_sub - t_base, 0.0) / (sum(frac) / len(frac)))      # exchange scaled to all pairs
    wall, dt = float(np.mean(walls)), float(np.mean(fulls))
    value = nb / dt
    sample = ("%d of %d walkers per step; exchange on %s of the i<=j pairs (stratified by |i-j|, own Jacobi factors), its time scaled to "
              "all pairs; Theta/one-body/Coulomb in full" % (nb, n_w, "+".join("%d/%d" % (len(f.r), len(oracle.all_pairs(o)[0])) for f, o in zip(fs, P.n_occ))))
    # ms_per_step is the wall time MEASURED per iteration (two oracle calls on the sample); `value` is an estimate for the
    # full pair list (the oracle's own SVD of every pair would take hours), hence "extrapolated": true.
    line = {"impl": "reference", "metric": METRIC, "value": round(value, 3), "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": round(wall * 1e3, 2), "extrapolated": True,
            "ms_per_step_all_pairs_estimate": round(dt * 1e3, 2),
            "extrapolation": "value = sample walkers / (t_noexchange + (t_sample - t_noexchange) * all pairs / sampled pairs)",
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cfg, reading, T, n_w), "N": P.N, "N_occ": list(P.n_occ)[:P.n_spin], "N_chol": int(P.L.shape[0]),
                       "N_w_per_gpu": n_w, "T_SVD": T},
            "cpu_baseline": {"value": round(value, 3), "unit": UNIT, "kind": "oracle", "cores": oracle.num_threads(), "sample": sample},
            "e2e": {"value": round(value, 3), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def run_cas_step(args):
    """--cas-step N_DET: multi-determinant local-energy steps alone, for ncu captures of the k_cas_*
    kernels: --walkers real walkers (default 400) of --config/--reading, 6 active virtuals, --cas-holes active occupied
    columns, excitation rank <= --cas-exc, mode --cas-mode; one JSON line."""
    import torch

    import gen
    import paper_2202_00832_b200 as lo
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    n_det, n_w, smw = args.cas_step, args.walkers or 400, args.cas_mode == "smw"
    P = gen.make_problem(args.config, reading=args.reading)
    T = args.threshold if args.threshold is not None else gen.CONFIGS[args.config].thresholds[0]
    Trs = [gen.make_cas_trial(P, n_virt=6, n_act_occ=args.cas_holes, n_det=n_det, max_exc=args.cas_exc, spin=s) for s in range(P.n_spin)]
    Tr = Trs[0]
    F = lo.Factors.setup(P.h, P.L, [t.C for t in Trs], T, device=0, max_walkers=n_w if smw else n_w * n_det, gpu_svd=True)
    F.set_cas_trial(Tr.n_ref, Tr.holes, Tr.parts, Tr.coef, n_w, smw_energy=smw)
    if P.n_spin == 2:                 # unrestricted trial: different alpha / beta strings
        F.set_cas_trial_beta(Trs[1].n_ref, Trs[1].holes, Trs[1].parts)
    phis = [torch.from_numpy(p).cuda() for p in gen.make_walkers(P, n_w)]
    phi = phis[0] if P.n_spin == 1 else phis
    call = (lambda: F.local_energy_cas(phi)) if P.n_spin == 1 else (lambda: F.local_energy_cas(phis[0], phis[1]))
    for _ in range(max(args.warmup, 1)):
        E, st = call()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        E, st = call()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    info = F.info()
    print(json.dumps({"cas_step": workload_name(args.config, args.reading, T, n_w), "mode": args.cas_mode, "n_det": n_det, "n_spin": P.n_spin,
                      "max_exc": args.cas_exc, "active_occupied": args.cas_holes, "tiles": info.n_tiles, "sum_rank": sum(info.sum_rank),
                      "ms_per_step": round(ms, 4), "energies_per_s": round(n_w / (ms * 1e-3), 2),
                      "determinant_energies_per_s": round(n_w * n_det / (ms * 1e-3), 2), "status_ok": bool((st == 0).all()),
                      "E_L0": [E[0, 0].real.item(), E[0, 0].imag.item()]}), flush=True)


def self_launch(n):
    """Re-run this command line under torch.distributed.run with n ranks on this node (rendezvous on 127.0.0.1, a free
    port); NCCL's INFO log stays on (stderr) so the rank count can be read off the run.  Returns the exit code."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")
    env.setdefault("OMP_NUM_THREADS", str(max(1, (os.cpu_count() or n) // n)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n), "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd, env=env)


def run_launch_check(args):
    """Bring up the ranks exactly as run_ours does (NCCL with one GPU per rank; gloo when the box has no GPU), take the
    max over ranks of a per-rank number and the sum of the ranks' walker counts, print one line on rank 0."""
    import torch
    import torch.distributed as dist

    from paper_2202_00832_b200.dist import max_over_ranks, sum_over_ranks
    rank, world, local = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1)), int(os.environ.get("LOCAL_RANK", 0))
    cuda = torch.cuda.is_available()
    dev = torch.device("cuda", local) if cuda else None
    if cuda:
        torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl" if cuda else "gloo", **({"device_id": dev} if cuda else {}))
        dist.barrier()
    ms = max_over_ranks(10.0 + rank, dev)
    total = sum_over_ranks(float(args.walkers or 1), dev)
    if rank == 0:
        print(json.dumps({"launch_check": True, "n_gpus": world, "backend": ("nccl" if cuda else "gloo") if world > 1 else None,
                          "max_ms": ms, "walkers_total": total}), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index (default 2: pentacene-sized, the headline)")
    ap.add_argument("--reading", default="element", choices=["element", "vector"])
    ap.add_argument("--exchange", default="int8", choices=["int8", "dmma"],
                    help="exchange route of the timed step: INT8 digit slices on tcgen05 (default; the DMMA route is timed beside it) or FP64 DMMA only")
    ap.add_argument("--threshold", type=float, default=None)
    ap.add_argument("--walkers", type=int, default=None)
    ap.add_argument("--cpu-walkers", type=int, default=192, help="walkers of the batch the oracle is timed on (cpu_baseline)")
    ap.add_argument("--ref-walkers", type=int, default=32)
    ap.add_argument("--ref-pairs", type=int, default=128)
    ap.add_argument("--no-propagator", dest="propagator", action="store_false",
                    help="skip the NEXT-1 propagator-formation measurement (reported under \"next\", never part of `value`)")
    ap.add_argument("--cas", type=int, default=0, help="also time the NEXT-2 multi-determinant path with this many determinants "
                    "(N_w / cas real walkers; reported under \"next\", never part of `value`)")
    ap.add_argument("--sweep", action="store_true", help="threshold sweep (BASELINE.json:configs[4]): one JSON line per threshold")
    ap.add_argument("--sweep-exact-walkers", type=int, default=4, help="walkers whose exact E_K the oracle computes in --sweep")
    ap.add_argument("--screen", action="store_true", help="pair-screening study on chains (NEXT-4): one JSON line per (chain length, cutoff)")
    ap.add_argument("--screen-sites", type=int, nargs="+", default=[20, 40, 80, 160])
    ap.add_argument("--screen-cutoffs", type=float, nargs="+", default=[0.0, 1e-6, 1e-4, 1e-2])
    ap.add_argument("--cas-step", type=int, default=0, help="run only multi-determinant steps with this many determinants (ncu target)")
    ap.add_argument("--cas-mode", default="smw", choices=["smw", "direct"])
    ap.add_argument("--cas-exc", type=int, default=4, help="maximum excitation rank of the synthetic CI expansion")
    ap.add_argument("--cas-holes", type=int, default=6, help="active occupied (hole) columns of the synthetic CI expansion")
    ap.add_argument("--launch-check", action="store_true", help="only bring up the N ranks (NCCL on GPUs, gloo without), reduce a dummy "
                    "timing over them and print {\"n_gpus\": N, ...}; exercises the --gpus N launcher without the workload")
    args = ap.parse_args()
    if args.gpus < 1:
        ap.error("--gpus must be >= 1")
    env_world = os.environ.get("WORLD_SIZE")
    if env_world is not None and int(env_world) != args.gpus and args.impl == "ours":
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%s; launch one rank per GPU (torchrun --nproc-per-node %d) or drop --gpus"
                         % (args.gpus, env_world, args.gpus))
    if env_world is None and args.gpus > 1 and args.impl == "ours" and not args.sweep:
        # `python bench.py --gpus N` without torchrun: start the N ranks here (one per GPU) and hand over
        sys.exit(self_launch(args.gpus))
    if args.launch_check:
        run_launch_check(args)
    elif args.cas_step > 0:
        run_cas_step(args)
    elif args.screen:
        run_screen(args)
    elif args.sweep:
        if args.config == 2 and "--config" not in " ".join(sys.argv):
            args.config = 4
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
