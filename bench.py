#!/usr/bin/env python
"""bench.py -- BASELINE.json's headline metric on its headline workload.

  metric    interactions/s of the full force sweep (every particle against every particle:
            acceleration + jerk + potential + nearest neighbour, double-single separations)
  workload  C4 of BASELINE.json: N = 1 048 576 equal-mass Plummer sphere, eps = 1e-4, synthetic
            (seeded generator, paper_0902_4463_b200/inputs.py)

One "step" = one pass of the whole hot path over the particle set:
  a-1 j-store update (all N particles re-sent: in a sweep every particle was "corrected"),
  a-2 predictor, a-3 i-block, a-4 force kernel, a-5 combine, a-6 results.
`value`  : inputs (fp64) already resident in HBM, results left in HBM  (g6x_*_dev entry points)
`e2e`    : the same step through the host entry points (g6x_set_j_particles, g6calc_firsthalf,
           g6calc_lasthalf2) with HOST buffers; H2D and D2H copies inside the timed region.

Multi-GPU (torchrun, one rank per GPU): the sweep is sharded over the i-particles -- every rank
holds and predicts all N j-particles and computes the forces on its N/G i-particles; no
data-path collective (SURVEY.md 8(e) option 2).  Total work is fixed => "scaling": "strong".

`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same
workload on the host cores.
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

WORKLOAD = "C4"
METRIC = "interactions/s (N=1048576 Plummer full force sweep: acc+jerk+pot+nearest neighbour, DS separations)"
# algorithmic work of one pairwise interaction
FP32_INSTR_PER_INTERACTION = 33      # FP32-pipe lane-instructions
FLOP47 = 47                          # same work counted as flops with FMA = 2
FLOP_PAPER = 60                      # the paper's convention (PAPER.md:164 fn.9); 66 with DS
SM_COUNT = 148
FP32_LANES_PER_SM = 128
SM_MAX_MHZ_FALLBACK = 1965.0


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "sm_max_mhz": SM_MAX_MHZ_FALLBACK}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled while the timed region runs."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index=0):
        self.gpu = gpu_index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            f = [s.strip() for s in line.split(",")]
            if len(f) >= 9:
                self.rows.append(f)

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        for f in self.rows:
            try:
                sm.append(float(f[1])); mx.append(float(f[2])); power.append(float(f[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        busy = [c for c, p in zip(sm, power) if p > 0.5 * max(power)] or sm
        return {"sm_mhz": float(np.median(busy)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                "power_w_max": float(max(power)), "samples": len(sm)}


class Probes:
    """bench.py's measurement aids (paper_0902_4463_b200/csrc/bench/g6_bench_probe.cu -> libg6b200_probe.so; not part of
    libg6b200, not on the path): FP32 instruction-rate probes, the production pair loop with ablations, a read-only pass."""
    FP32_MODES = ((0, "scalar_ffma_x_d_acc_reuse"), (1, "scalar_ffma_three_changing_sources"), (2, "ffma2_two_distinct_pairs"),
                  (3, "ffma2_two_pairs_plus_reused"), (4, "ffma2_three_distinct_pairs"), (5, "ffma2_two_pairs_plus_32bit_broadcast"),
                  (6, "fmul2_one_pair_alternating_ffma2_three_pairs"), (7, "fadd2_fmul2_ffma2_mix_one_changing_source"))
    PAIR_VARIANTS = ((0, "production_pair2_ds_newton"), (1, "pure_fp32_separations"), (2, "three_operand_ffma2_made_two_operand"),
                     (3, "no_nearest_neighbour_tracking"))

    def __init__(self):
        import ctypes as C
        from paper_0902_4463_b200 import build
        self.C = C
        self.L = C.CDLL(build.build_probe())

    def fp32_rate(self, mode, ctas_per_sm, stream=0):
        r = self.C.c_double(0.0)
        rc = self.L.g6p_fp32_rate(self.C.c_int(mode), self.C.c_int(ctas_per_sm), self.C.c_void_p(stream), self.C.byref(r))
        if rc:
            raise RuntimeError(f"g6p_fp32_rate failed: cudaError {rc}")
        return r.value

    def pair_rate(self, ab, shape, stream=0):
        r = self.C.c_double(0.0)
        rc = self.L.g6p_pair_rate(self.C.c_int(ab), self.C.c_int(shape), self.C.c_void_p(stream), self.C.byref(r))
        if rc:
            raise RuntimeError(f"g6p_pair_rate failed: cudaError {rc}")
        return r.value

    def read_pass(self, tensor, stream):
        nbytes = tensor.numel() * tensor.element_size() // 16 * 16
        rc = self.L.g6p_read_pass(self.C.c_void_p(tensor.data_ptr()), self.C.c_ulonglong(nbytes), self.C.c_void_p(stream))
        if rc:
            raise RuntimeError(f"g6p_read_pass failed: cudaError {rc}")

    MIX_KINDS = ((1, "lds"), (2, "mov_imm"), (3, "iadd"), (4, "lop3_two_reads"), (5, "fmnmx"), (6, "fmnmx3"), (7, "vimnmx3"),
                 (8, "scalar_ffma"), (9, "mufu_rsq"))
    OPERAND_MODES = ((0, "ffma2_acc_x_shared_vector_pair_reuse"), (1, "ffma2_acc_x_uniform_register_pair"), (2, "ffma2_acc_x_32bit_broadcast"),
                     (3, "fadd2_acc_shared_vector_pair"), (4, "fadd2_acc_uniform_register_pair"), (5, "ffma2_three_distinct_vector_pairs"))

    def mix_cycles(self, kind, extra, sm_hz, stream=0):
        r = self.C.c_double(0.0)
        rc = self.L.g6p_mix_cycles(self.C.c_int(kind), self.C.c_int(extra), self.C.c_double(sm_hz), self.C.c_void_p(stream), self.C.byref(r))
        if rc:
            raise RuntimeError(f"g6p_mix_cycles failed: cudaError {rc}")
        return r.value

    def operand_rate(self, mode, stream=0):
        r = self.C.c_double(0.0)
        rc = self.L.g6p_operand_rate(self.C.c_int(mode), self.C.c_void_p(stream), self.C.byref(r))
        if rc:
            raise RuntimeError(f"g6p_operand_rate failed: cudaError {rc}")
        return r.value

    def pair_rate_cbank(self, shape, stream=0):
        r = self.C.c_double(0.0)
        rc = self.L.g6p_pair_rate_cbank(self.C.c_int(shape), self.C.c_void_p(stream), self.C.byref(r))
        if rc:
            raise RuntimeError(f"g6p_pair_rate_cbank failed: cudaError {rc}")
        return r.value

    def extended(self, peak_inst, sm_hz, stream=0):
        """--probes only (profiles/r02_fp32_operand_probes.md): what one non-FMA instruction costs next to a saturated FFMA2 stream,
        which operand forms cost no vector-register read, and the pair loop with its j-tiles in the constant bank"""
        out = {}
        base = self.mix_cycles(0, 0, sm_hz, stream)
        mix = {"twelve_ffma2_alone_cycles": base}
        for kind, name in self.MIX_KINDS:
            row = {}
            for extra in ((1, 2, 4) if name == "mufu_rsq" else (4, 12)):
                c = self.mix_cycles(kind, extra, sm_hz, stream)
                row[f"plus_{extra}"] = {"cycles": c, "cost_each": (c - base) / extra}
            mix[name] = row
        out["non_fma_instruction_next_to_12_ffma2"] = mix
        out["operand_forms_frac_of_peak"] = {name: self.operand_rate(mode, stream) / peak_inst for mode, name in self.OPERAND_MODES}
        cb = {sh: self.pair_rate_cbank(k, stream) for k, sh in ((0, "128x2"), (1, "128x1"))}
        out["pair_loop_j_tiles_in_constant_bank"] = {"interactions_per_s": cb, "pipe_busy_frac": {k: v * 36 / peak_inst for k, v in cb.items()},
                                                     "frac_of_peak_at_33": {k: v * 33 / peak_inst for k, v in cb.items()}}
        return out

    def table(self, peak_inst, stream=0):
        """every probe as a fraction of the nominal FP32 peak (lane-instructions / s)"""
        out = {"fp32_instruction_streams_frac_of_peak": {}, "pair_loop": {}}
        for w in range(3):
            self.fp32_rate(2, 4, stream)                                    # bring the clocks up
        for mode, name in self.FP32_MODES:
            out["fp32_instruction_streams_frac_of_peak"][name] = max(self.fp32_rate(mode, c, stream) for c in (2, 4, 8)) / peak_inst
        for ab, name in self.PAIR_VARIANTS:
            per_pair = {0: 36, 1: 30, 2: 37, 3: 36.5}[ab]                  # packed FP32 instructions per pair evaluation of the variant (counted in its SASS)
            r = {sh: self.pair_rate(ab, k, stream) for k, sh in ((0, "128x2"), (1, "256x1"))}
            out["pair_loop"][name] = {"interactions_per_s": r, "fp32_instr_per_interaction_executed": per_pair,
                                      "pipe_busy_frac": {k: v * per_pair / peak_inst for k, v in r.items()},
                                      "frac_of_peak_at_33": {k: v * 33 / peak_inst for k, v in r.items()}}
        return out


def cpu_oracle_rate(x, v, m, eps2, idx, target_s, seed=7):
    """interactions/s of the oracle (as it stands) on a bounded sample of rows of the sweep."""
    from oracle import oracle as orc
    n = len(m)
    rng = np.random.default_rng(seed)
    probe = np.sort(rng.choice(n, 64, replace=False))
    t0 = time.perf_counter()
    orc.force(idx[probe], x[probe], v[probe], idx, x, v, m, eps2)
    dt = time.perf_counter() - t0
    rows = int(min(n, max(64, 64 * target_s / max(dt, 1e-3))))
    rows = max(orc.threads(), rows)
    sel = np.sort(rng.choice(n, rows, replace=False))
    t0 = time.perf_counter()
    orc.force(idx[sel], x[sel], v[sel], idx, x, v, m, eps2)
    dt = time.perf_counter() - t0
    return rows * float(n) / dt, rows, dt, orc.threads()


NI_SWEEP = (1, 16, 256, 4096, 65536)


def ni_sweep(g6, inputs, torch, dev, stream, flush, x, v, idx_all, n, eps2, peaks, probes, reps=10):
    """C4's block-step regime (BASELINE.json configs[3]): random active blocks of n_i particles
    against all N_j, one block step = predictor over all j (t_i changes every step) + force +
    combine.  Device times from CUDA events on the launching stream; `cold` = L2 flushed before
    every step, `warm` = back to back (the j-store and the predicted tiles stay in the 126 MB L2).
    Algorithmic bytes per step: 76 B/j when the predictor is fused into the
    force pass, else 76 + 40 (predictor) + 40 (force read) = 156 B/j."""
    f64 = torch.float64
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    sm_max = float(peaks.get("sm_max_mhz", SM_MAX_MHZ_FALLBACK))
    peak_inst = SM_COUNT * FP32_LANES_PER_SM * sm_max * 1e6
    rows = []
    # floor of a block step at small n_i: a kernel that only reads the j-store once (same bytes, L2 flushed)
    bare = []
    jstore_sized = torch.zeros(n * 76 // 4, dtype=torch.float32, device=dev)      # as many bytes as the raw j-store of n particles
    for k in range(reps + 3):
        flush.zero_()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record(stream); probes.read_pass(jstore_sized, stream.cuda_stream); e1.record(stream)
        torch.cuda.synchronize()
        if k >= 3:
            bare.append(e0.elapsed_time(e1) * 1e3)
    bare_us = float(np.median(bare))
    for ni in NI_SWEEP:
        if ni > n:
            continue
        block = inputs.active_subset(n, ni, 4040 + ni)
        to = lambda a, dt=f64: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dt)
        d_xi, d_vi, d_ii = to(x[block]), to(v[block]), to(idx_all[block], torch.int32)
        d_acc = torch.empty(ni, 3, dtype=f64, device=dev); d_jerk = torch.empty_like(d_acc)
        d_pot = torch.empty(ni, dtype=f64, device=dev); d_nn = torch.empty(ni, dtype=torch.int32, device=dev)
        d_r2 = torch.empty_like(d_pot)
        res = {}
        for mode in ("cold", "warm"):
            tot, frc, prd, cmb = [], [], [], []
            # pass 1: the library's per-phase events (they cost ~10 us of stream time per call); pass 2: timers off,
            # the step as a host code sees it (CUDA events around the call on the launching stream)
            for timers in (1, 0):
                g6.g6x_set_option(0, "timers", timers)
                for k in range(reps + 3):
                    if mode == "cold":
                        flush.zero_()
                    g6.g6_set_ti(0, (k % 2) * 2.0 ** -30)            # a new block time: the predictor runs again
                    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                    e0.record(stream)
                    g6.g6x_calc_dev(0, n, ni, d_ii, d_xi, d_vi, eps2, d_acc, d_jerk, d_pot, d_nn, d_r2)
                    e1.record(stream)
                    torch.cuda.synchronize()
                    if k < 3:
                        continue
                    if timers:
                        tm = g6.g6x_get_timers(0)
                        frc.append(tm["force_us"]); prd.append(tm["predict_us"]); cmb.append(tm["combine_us"])
                    else:
                        tot.append(e0.elapsed_time(e1) * 1e3)
            g6.g6x_set_option(0, "timers", 1)
            res[mode] = dict(step_us=float(np.median(tot)), force_us=float(np.median(frc)), predict_us=float(np.median(prd)),
                             combine_us=float(np.median(cmb)), jsplits=tm["jsplits"], ctas=tm["force_ctas"])
        fused = g6.g6x_get_option(0, "last_kernel") == 3          # the block-step kernel took the call (n_i <= 64)
        bytes_step = n * (76 if fused else 156)
        c = res["cold"]
        rows.append({"n_i": ni, "cold": res["cold"], "warm": res["warm"], "fused_predictor": bool(fused),
                     "interactions_per_s_cold": ni * float(n) / (c["step_us"] * 1e-6),
                     "interactions_per_s_warm": ni * float(n) / (res["warm"]["step_us"] * 1e-6),
                     "algorithmic_bytes_per_step": bytes_step,
                     "bare_read_us": bare_us, "step_over_bare_read": c["step_us"] / bare_us,
                     "hbm_gbs_cold": bytes_step / (c["step_us"] * 1e-6) / 1e9,
                     "hbm_frac_cold": bytes_step / (c["step_us"] * 1e-6) / 1e9 / hbm,
                     "fp32_frac_force_kernel_cold": FP32_INSTR_PER_INTERACTION * ni * float(n) / (c["force_us"] * 1e-6) / peak_inst})
    g6.g6_set_ti(0, 0.0)
    return rows


def neighbour_list_cost(g6, inputs, torch, dev, x, v, idx_all, n, eps2, ni=65536, reps=3):
    """What building neighbour lists costs (the paper: "a few tens of percent"): the same
    65536-block against all N_j with and without lists; h2_i = (2 x the local mean spacing)^2 of the
    Plummer model, i.e. ~30 neighbours per particle."""
    f64 = torch.float64
    ni = min(ni, n)
    block = inputs.active_subset(n, ni, 4040 + ni)
    to = lambda a, dt=f64: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dt)
    a = 3 * np.pi / 16
    r = np.linalg.norm(x[block], axis=1)
    rho = 3 / (4 * np.pi * a ** 3) * (1 + (r / a) ** 2) ** -2.5 * n
    h2 = (2.0 * rho ** (-1.0 / 3)) ** 2
    d_xi, d_vi, d_ii, d_h2 = to(x[block]), to(v[block]), to(idx_all[block], torch.int32), to(h2)
    d_acc = torch.empty(ni, 3, dtype=f64, device=dev); d_jerk = torch.empty_like(d_acc)
    d_pot = torch.empty(ni, dtype=f64, device=dev); d_nn = torch.empty(ni, dtype=torch.int32, device=dev); d_r2 = torch.empty_like(d_pot)
    maxlen = g6.g6x_get_option(0, "nb_maxlen")
    d_cnt = torch.zeros(ni, dtype=torch.int32, device=dev); d_lst = torch.empty(ni, maxlen, dtype=torch.int32, device=dev)
    g6.g6_set_ti(0, 0.0)
    out = {}
    for name in ("without", "with"):
        ts = []
        for k in range(reps + 1):
            if name == "with":
                g6.g6x_calc_dev_nb(0, n, ni, d_ii, d_xi, d_vi, eps2, d_acc, d_jerk, d_pot, d_nn, d_r2, d_h2, d_cnt, d_lst)
            else:
                g6.g6x_calc_dev(0, n, ni, d_ii, d_xi, d_vi, eps2, d_acc, d_jerk, d_pot, d_nn, d_r2)
            torch.cuda.synchronize()
            tm = g6.g6x_get_timers(0)
            if k > 0:
                ts.append(tm["force_us"] + tm["combine_us"])
        out[name] = float(np.median(ts))
    cnt = d_cnt.cpu().numpy()
    return {"n_i": ni, "force_plus_combine_us_without": out["without"], "force_plus_combine_us_with": out["with"],
            "cost": out["with"] / out["without"] - 1.0, "mean_neighbours": float(cnt.mean()), "max_neighbours": int(cnt.max()),
            "overflowed": int((cnt > maxlen).sum()), "nb_maxlen": maxlen}


def recorded_traffic(nj, ni, jsplits):
    """DRAM bytes of one force-kernel launch from the committed ncu capture, if it was taken on this configuration."""
    p = os.path.join(ROOT, "profiles", "r02_force_fast_traffic.json")
    try:
        rec = json.load(open(p))
    except Exception:
        return None
    if rec.get("n_j") == nj and rec.get("n_i") == ni and rec.get("jsplits") == jsplits:
        return int(rec["dram_bytes_read"]) + int(rec["dram_bytes_write"])
    return None


def double_single_cost(g6, inputs, torch, dev, x, v, idx_all, n, eps2, ni=65536, reps=3):
    """What the double-single separations cost (the paper: "<~ 20 %"): the same 65536-block against all N_j
    with option ds = 1 (Eq. 3: 9 packed adds per pair) and ds = 0 (pure FP32: 3 packed adds; lo words dropped by the predictor)."""
    f64 = torch.float64
    ni = min(ni, n)
    block = inputs.active_subset(n, ni, 4040 + ni)
    to = lambda a, dt=f64: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dt)
    d_xi, d_vi, d_ii = to(x[block]), to(v[block]), to(idx_all[block], torch.int32)
    d_acc = torch.empty(ni, 3, dtype=f64, device=dev); d_jerk = torch.empty_like(d_acc)
    d_pot = torch.empty(ni, dtype=f64, device=dev); d_nn = torch.empty(ni, dtype=torch.int32, device=dev); d_r2 = torch.empty_like(d_pot)
    g6.g6_set_ti(0, 0.0)
    out = {}
    for ds in (1, 0):
        g6.g6x_set_option(0, "ds", ds)
        ts = []
        for k in range(reps + 1):
            g6.g6x_calc_dev(0, n, ni, d_ii, d_xi, d_vi, eps2, d_acc, d_jerk, d_pot, d_nn, d_r2)
            torch.cuda.synchronize()
            if k > 0:
                ts.append(g6.g6x_get_timers(0)["force_us"])
        out[ds] = float(np.median(ts))
    g6.g6x_set_option(0, "ds", 1)
    return {"n_i": ni, "force_us_double_single": out[1], "force_us_pure_fp32": out[0], "cost": out[1] / out[0] - 1.0,
            "interactions_per_s_double_single": ni * float(n) / (out[1] * 1e-6), "interactions_per_s_pure_fp32": ni * float(n) / (out[0] * 1e-6)}


def c3_sweep(g6, inputs, torch, dev, peaks, reps=5):
    """BASELINE.json configs[2] (C3): full force sweep at N = 131072, device-resident, L2-resident j-store
    (a side figure; the headline is C4).  Replaces the j-store contents: call last."""
    f64 = torch.float64
    x, v, m, eps2 = inputs.config("C3")
    n = len(m)
    to = lambda a, dt=f64: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dt)
    d_x, d_v, d_m, d_idx = to(x), to(v), to(m), to(np.arange(n, dtype=np.int32), torch.int32)
    z3 = torch.zeros(n, 3, dtype=f64, device=dev); zt = torch.zeros(n, dtype=f64, device=dev)
    acc = torch.empty(n, 3, dtype=f64, device=dev); jerk = torch.empty_like(acc); pot = torch.empty(n, dtype=f64, device=dev)
    nn = torch.empty(n, dtype=torch.int32, device=dev); r2 = torch.empty_like(pot)
    ts, fs = [], []
    for k in range(reps + 2):
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record(torch.cuda.current_stream())
        g6.g6x_set_j_particles_dev(0, 0, n, d_idx, zt, d_m, z3, z3, d_v, d_x)
        g6.g6_set_ti(0, 0.0)
        g6.g6x_calc_dev(0, n, n, d_idx, d_x, d_v, eps2, acc, jerk, pot, nn, r2)
        e1.record(torch.cuda.current_stream())
        torch.cuda.synchronize()
        if k >= 2:
            ts.append(e0.elapsed_time(e1)); fs.append(g6.g6x_get_timers(0)["force_us"])
    ms, f_us = float(np.median(ts)), float(np.median(fs))
    peak_inst = SM_COUNT * FP32_LANES_PER_SM * float(peaks.get("sm_max_mhz", SM_MAX_MHZ_FALLBACK)) * 1e6
    return {"workload": f"C3: N={n} equal-mass Plummer, eps=1e-4, full sweep", "ms_per_step": ms, "interactions_per_s": float(n) * n / (ms * 1e-3),
            "gflops_60": FLOP_PAPER * float(n) * n / (ms * 1e-3) / 1e9, "force_kernel_ms": f_us / 1e3,
            "fp32_frac_force_kernel": FP32_INSTR_PER_INTERACTION * float(n) * n / (f_us * 1e-6) / peak_inst}


def c2_hermite(g6, inputs, t_end=1.0):
    """BASELINE.json configs[1] (C2): N = 32768 equal-mass Plummer, eps = 1e-4, 4th-order Hermite with block time steps (eta = 0.01,
    power-of-two steps) to t = 1, with the device-resident driver (g6hd_*: the block-step loop as one persistent kernel, blocks above
    768 particles through the sweep path).  A side figure: wall time of g6hd_evolve and the block-size histogram; the energy drift is
    the parity suite's business (tests/test_hermite_gpu.py::test_c2_full_run_vs_oracle_driven).  Replaces the j-store contents: call last."""
    x, v, m, eps2 = inputs.config("C2")
    t0 = time.perf_counter()
    h = g6.HermiteDev(0, x, v, m, eps2, 0.01)
    t_init = time.perf_counter() - t0
    try:
        t0 = time.perf_counter()
        h.evolve(t_end)
        wall = time.perf_counter() - t0
        st = h.stats()
    finally:
        h.close()
    return {"workload": f"C2: N={len(m)} equal-mass Plummer, eps=1e-4, Hermite block time steps eta=0.01, t=0..{t_end:g}", "driver": "device-resident (g6hd_*)",
            "wall_s": wall, "init_s": t_init, "block_steps": st["n_block_steps"], "particle_steps": st["n_particle_steps"],
            "us_per_block_step": 1e6 * wall / max(1, st["n_block_steps"]), "interactions": st["interactions"],
            "interactions_per_s": st["interactions"] / wall, "gflops_60": FLOP_PAPER * st["interactions"] / wall / 1e9,
            "dt_min": st["dt_min"], "ni_hist_log2": [int(c) for c in st["ni_hist_log2"][:17]]}


def bench_config(inputs, n, eps2, newton, world):
    """the `config` object of the BENCH line: the same for the CUDA arm and for --impl reference"""
    return {"workload": f"{WORKLOAD}: N={n} equal-mass Plummer sphere, eps=1e-4, full force sweep n_i=N_j=N",
            "n": n, "eps2": eps2, "seed": inputs.CONFIGS[WORKLOAD]["seed"], "newton_step": int(newton),
            "parallelism": f"i-split x{world}" if world > 1 else "1 GPU", "l2": "flushed between timed steps (512 MiB write)"}


def run_reference(args):
    """--impl reference: the oracle, timed on the host cores on a bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as orc
    from paper_0902_4463_b200 import inputs
    orc.build(False)
    x, v, m, eps2 = inputs.config(WORKLOAD, n=args.n)
    n = len(m)
    idx = np.arange(n, dtype=np.int32)
    rng = np.random.default_rng(11)
    # size one step to ~args.ref_seconds of CPU work
    probe = np.sort(rng.choice(n, 64, replace=False))
    t0 = time.perf_counter(); orc.force(idx[probe], x[probe], v[probe], idx, x, v, m, eps2); dt = time.perf_counter() - t0
    rows = int(min(n, max(orc.threads(), 64 * args.ref_seconds / max(dt, 1e-3))))
    times = []
    for step in range(args.warmup + args.steps):
        sel = np.sort(rng.choice(n, rows, replace=False))
        t0 = time.perf_counter()
        orc.force(idx[sel], x[sel], v[sel], idx, x, v, m, eps2)
        if step >= args.warmup:
            times.append(time.perf_counter() - t0)
    total = sum(times)
    value = args.steps * rows * float(n) / total
    sample = f"{rows} randomly chosen i-rows x all {n} j per step (a bounded sample of the sweep), {args.steps} steps"
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": "interactions/s", "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "strong",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           # the same config as the CUDA arm's line (the driver compares them); that each step is a bounded sample of the rows is
           # said in cpu_baseline.sample
           "config": bench_config(inputs, n, eps2, 1 if args.newton is None else int(args.newton), max(1, args.gpus)),
           "cpu_baseline": {"value": value, "unit": "interactions/s", "cores": orc.threads(), "kind": "oracle", "sample": sample},
           "e2e": {"value": value, "unit": "interactions/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gflops_60": value * FLOP_PAPER / 1e9}
    print(json.dumps(out), flush=True)


def run_jsplit(args, torch, dist, g6, inputs, world, rank, local, dev):
    """--mode jsplit: one block step of n_i particles under the paper's multi-GPU scheme: rank r holds the
    j-particles of addresses [r N/G, (r+1) N/G), every rank computes partial forces on the SAME i-block (predictor over its
    slice + force + combine), then two allreduces (MIN on the nearest-neighbour keys, SUM on acc | jerk | pot | index) over
    NCCL, stream-ordered with the kernels (sharding.JSplit).  value = n_i x N interactions per step over the max-over-ranks
    time; at G = 1 the collectives are no-ops and the line is the single-GPU block step."""
    from paper_0902_4463_b200.sharding import JSplit, LibOps, j_range
    x, v, m, eps2 = inputs.config(WORKLOAD, n=args.n)
    n = len(m)
    idx = np.arange(n, dtype=np.int32)
    ni = min(args.ni, n)
    j0, j1 = j_range(rank, world, n)
    f64 = torch.float64
    to = lambda a, dt=f64: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dt)
    g6.g6_open(0)
    g6.g6x_set_npipes(1 << 21)
    stream = torch.cuda.Stream(device=dev)
    torch.cuda.set_stream(stream)
    ops = LibOps(0)                                      # moves the cluster onto torch's current stream
    nl = j1 - j0
    z3 = torch.zeros(nl, 3, dtype=f64, device=dev)
    g6.g6x_set_j_particles_dev(0, 0, nl, to(idx[j0:j1], torch.int32), torch.zeros(nl, dtype=f64, device=dev), to(m[j0:j1]), z3, z3,
                               to(v[j0:j1]), to(x[j0:j1]))
    block = inputs.active_subset(n, ni, 4040 + ni)
    d_ii, d_xi, d_vi = to(idx[block], torch.int32), to(x[block]).reshape(-1), to(v[block]).reshape(-1)
    js = JSplit(ops, rank, world) if world > 1 else JSplit(ops, 0, 1, allreduce=lambda t, op: None)
    flush = torch.empty(512 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def step(k):
        g6.g6_set_ti(0, (k % 2) * 2.0 ** -30)            # a new block time: the predictor runs again, as in a block step
        return js.calc(nl, ni, d_ii, d_xi, d_vi, eps2)

    for k in range(max(args.warmup, 3)):
        flush.zero_()
        step(k)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for k in range(args.steps):
        flush.zero_()
        barrier()
        ev[k][0].record(stream)
        step(k)
        ev[k][1].record(stream)
    barrier()
    clocks = sampler.stop()
    t_ms = torch.tensor([sum(a.elapsed_time(b) for a, b in ev)], dtype=f64, device=dev)
    if world > 1:
        dist.all_reduce(t_ms, op=dist.ReduceOp.MAX)
    ms_total = float(t_ms.item())
    if rank == 0:
        value = args.steps * float(ni) * float(n) / (ms_total * 1e-3)
        print(json.dumps({"metric": "interactions/s (one block step of n_i particles against N j-particles split over the GPUs, PAPER.md:122)",
                          "value": value, "unit": "interactions/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
                          "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                          "dtype": "f32 (double-single separations, fp64 accumulation across tiles)", "data": "synthetic",
                          "config": {"workload": f"{WORKLOAD}: N={n} equal-mass Plummer sphere, eps=1e-4, block of n_i={ni} random active particles, j-split x{world}",
                                     "n": n, "n_i": ni, "parallelism": f"j-split x{world}: 2 allreduces per step (8 B + 64 B per i-particle)",
                                     "l2": "flushed between timed steps (512 MiB write)"},
                          "clocks": clocks, "gflops_60": value * FLOP_PAPER / 1e9, "gpu_launches": 6 * args.steps}), flush=True)
    g6.g6_close(0)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=None, help="override N (same seed) for quick checks; the headline is the default")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="CPU work of the cpu_baseline leg")
    ap.add_argument("--ref-seconds", type=float, default=8.0, help="CPU work per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-sweep", action="store_true", help="skip the C4 n_i sweep (block-step regime)")
    ap.add_argument("--newton", type=int, default=None, help="override the library default (1 = rsqrt + one Newton step)")
    ap.add_argument("--probes", action="store_true", help="only run the FP32 operand-bandwidth and pair-loop probes and print their table")
    ap.add_argument("--mode", default="sweep", choices=["sweep", "jsplit"],
                    help="sweep: the headline (i-split under torchrun); jsplit: the paper's multi-GPU scheme (PAPER.md:122), every rank "
                         "holds N/G j-particles and all ranks compute the same block of --ni i-particles, partial forces allreduced")
    ap.add_argument("--ni", type=int, default=4096, help="block size of --mode jsplit (n_i <= 4096 is the regime it is for)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = max(args.warmup, 0)
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_0902_4463_b200 import build, g6, inputs
    from paper_0902_4463_b200.sharding import i_range

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    os.environ["G6_DEVICE"] = str(local)
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()

    if args.probes:
        if rank == 0:
            peaks, _ = measured_peaks()
            peak_inst = SM_COUNT * FP32_LANES_PER_SM * float(peaks.get("sm_max_mhz", SM_MAX_MHZ_FALLBACK)) * 1e6
            pr = Probes()
            sm_hz = float(peaks.get("sm_max_mhz", SM_MAX_MHZ_FALLBACK)) * 1e6
            print(json.dumps({"probes": pr.table(peak_inst), "probes_extended": pr.extended(peak_inst, sm_hz), "peak_lane_instr_per_s": peak_inst,
                              "sm_hz_assumed": sm_hz}), flush=True)
        return
    if args.mode == "jsplit":
        return run_jsplit(args, torch, dist, g6, inputs, world, rank, local, dev)

    x, v, m, eps2 = inputs.config(WORKLOAD, n=args.n)
    n = len(m)
    idx = np.arange(n, dtype=np.int32)
    i0, i1 = i_range(rank, world, n)
    ni = i1 - i0

    g6.g6_open(0)
    g6.g6x_set_npipes(1 << 21)
    g6.g6x_set_option(0, "timers", 1)                # per-phase CUDA events on the library's stream (off by default)
    if args.newton is not None:
        g6.g6x_set_option(0, "newton", args.newton)
    newton = g6.g6x_get_option(0, "newton")
    stream = torch.cuda.Stream(device=dev)             # a real (non-default) stream: handle != 0
    torch.cuda.set_stream(stream)
    g6.g6x_set_stream(0, stream.cuda_stream)          # so that torch events bracket the library's kernels

    f64 = torch.float64
    to = lambda a, dt=f64: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dt)
    d_x, d_v, d_m, d_idx = to(x), to(v), to(m), to(idx, torch.int32)
    d_t = torch.zeros(n, dtype=f64, device=dev); d_z3 = torch.zeros(n, 3, dtype=f64, device=dev)
    d_xi, d_vi, d_ii = d_x[i0:i1].contiguous(), d_v[i0:i1].contiguous(), d_idx[i0:i1].contiguous()
    d_acc = torch.empty(ni, 3, dtype=f64, device=dev); d_jerk = torch.empty_like(d_acc)
    d_pot = torch.empty(ni, dtype=f64, device=dev); d_nn = torch.empty(ni, dtype=torch.int32, device=dev); d_r2 = torch.empty_like(d_pot)
    flush = torch.empty(512 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)      # 512 MiB > 126 MB L2

    # multi-GPU (i-split): the shards meet -- every rank ends the step with ALL n rows of results, gathered over NCCL
    # (one all_gather of 72 B per i-particle) inside the timed region
    ni_pad = -(-n // world)
    if world > 1:
        d_rows = torch.zeros(ni_pad, 9, dtype=f64, device=dev)           # acc | jerk | pot | nn_r2 | nn_index (exact in fp64)
        d_all = torch.empty(world * ni_pad, 9, dtype=f64, device=dev)

    def step_dev():
        g6.g6x_set_j_particles_dev(0, 0, n, d_idx, d_t, d_m, d_z3, d_z3, d_v, d_x)       # a-1
        g6.g6_set_ti(0, 0.0)
        g6.g6x_calc_dev(0, n, ni, d_ii, d_xi, d_vi, eps2, d_acc, d_jerk, d_pot, d_nn, d_r2)   # a-2 .. a-5
        if world > 1:                                     # same stream as the library's kernels: stream-ordered, no host sync
            d_rows[:ni, 0:3] = d_acc; d_rows[:ni, 3:6] = d_jerk; d_rows[:ni, 6] = d_pot; d_rows[:ni, 7] = d_r2; d_rows[:ni, 8] = d_nn
            dist.all_gather_into_tensor(d_all, d_rows)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        flush.zero_()
        step_dev()
    barrier()

    sampler = ClockSampler(local)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    force_us, pred_us, comb_us = [], [], []
    barrier()
    wall0 = time.perf_counter()
    for k in range(args.steps):
        flush.zero_()                                     # L2 flush between timed iterations (outside the events)
        ev[k][0].record(stream)
        step_dev()
        ev[k][1].record(stream)
        torch.cuda.synchronize()
        tm = g6.g6x_get_timers(0)                         # the library's own CUDA events, same stream
        force_us.append(tm["force_us"]); pred_us.append(tm["predict_us"]); comb_us.append(tm["combine_us"])
    barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    ms = sum(a.elapsed_time(b) for a, b in ev)
    t_ms = torch.tensor([ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t_ms, op=dist.ReduceOp.MAX)
    ms_total = float(t_ms.item())
    value = args.steps * float(n) * float(n) / (ms_total * 1e-3)

    # ---- end to end through the host entry points (rank-local shard, host buffers) ------------------
    e2e = None
    if not args.no_e2e:
        z3 = np.zeros((n, 3)); tz = np.zeros(n)
        xi_h, vi_h, ii_h = np.ascontiguousarray(x[i0:i1]), np.ascontiguousarray(v[i0:i1]), np.ascontiguousarray(idx[i0:i1])

        host_group = dist.new_group(backend="gloo") if world > 1 else None
        rows_h = torch.zeros(ni_pad, 8, dtype=f64)
        all_h = [torch.empty_like(rows_h) for _ in range(world)]

        def step_host():
            g6.g6x_set_j_particles(0, 0, idx, tz, m, z3, z3, v, x)
            g6.g6_set_ti(0, 0.0)
            g6.g6calc_firsthalf(0, n, ni, ii_h, xi_h, vi_h, eps2=eps2)
            acc_h, jerk_h, pot_h, nn_h = g6.g6calc_lasthalf2(0, n, ni, eps2=eps2)
            if world > 1:                                 # the shards meet on the host too (host arrays in, host arrays out)
                rows_h[:ni, 0:3] = torch.from_numpy(acc_h); rows_h[:ni, 3:6] = torch.from_numpy(jerk_h)
                rows_h[:ni, 6] = torch.from_numpy(pot_h); rows_h[:ni, 7] = torch.from_numpy(nn_h.astype(np.float64))
                dist.all_gather(all_h, rows_h, group=host_group)
            return acc_h, jerk_h, pot_h, nn_h
        step_host()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            flush.zero_()
            torch.cuda.synchronize()
            r = step_host()
        barrier()
        e2e_s = time.perf_counter() - t0
        t_e = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t_e, op=dist.ReduceOp.MAX)
        h2d = (x.nbytes + v.nbytes + 2 * z3.nbytes + tz.nbytes + m.nbytes + idx.nbytes) + (xi_h.nbytes + vi_h.nbytes + ii_h.nbytes)
        d2h = ni * (3 * 8 + 3 * 8 + 8 + 4 + 8)
        e2e = {"value": args.steps * float(n) * float(n) / float(t_e.item()), "unit": "interactions/s",
               "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "note": "host arrays in, host arrays out (library stages through its own pinned buffers); includes the L2 flush"}

    sweep = None
    c3 = None
    c2 = None
    nb_cost = None
    ceilings = None
    ds_cost = None
    probes = Probes() if rank == 0 else None
    if rank == 0 and world == 1 and not args.no_sweep:
        sweep = ni_sweep(g6, inputs, torch, dev, stream, flush, x, v, idx, n, eps2, measured_peaks()[0], probes)
        nb_cost = neighbour_list_cost(g6, inputs, torch, dev, x, v, idx, n, eps2)
        ds_cost = double_single_cost(g6, inputs, torch, dev, x, v, idx, n, eps2)
        c3 = c3_sweep(g6, inputs, torch, dev, measured_peaks()[0]) if args.n is None else None
        c2 = c2_hermite(g6, inputs) if args.n is None else None
    if rank == 0:
        # what the FP32 pipes sustain for register-sourced instruction streams and for the pair loop itself (libg6b200_probe.so), live
        ceilings = probes.table(SM_COUNT * FP32_LANES_PER_SM * float(measured_peaks()[0].get("sm_max_mhz", SM_MAX_MHZ_FALLBACK)) * 1e6, stream.cuda_stream)

    if rank == 0:
        peaks, peaks_src = measured_peaks()
        sm_max = float(peaks.get("sm_max_mhz", SM_MAX_MHZ_FALLBACK))
        peak_inst = SM_COUNT * FP32_LANES_PER_SM * sm_max * 1e6                 # FP32 lane-instructions / s
        f_us = float(np.mean(force_us))
        inter_per_launch = float(ni) * float(n)
        ach_inst = FP32_INSTR_PER_INTERACTION * inter_per_launch / (f_us * 1e-6)
        roofline = {"bound": "alu", "kernel": "k_force_fast",
                    "achieved": 2 * ach_inst / 1e12, "peak": 2 * peak_inst / 1e12,
                    "unit": "TFLOP/s", "frac": ach_inst / peak_inst,
                    # dram__bytes_read.sum + dram__bytes_write.sum of one launch of this kernel from the committed ncu --set full capture
                    # (profiles/r02_force_fast_traffic.json names it); null unless that capture had this run's n_j, n_i and j-split count
                    "traffic": recorded_traffic(n, ni, int(tm["jsplits"])),
                    "how": ("FP32-pipe issue-slot equivalent: 33 algorithmic FP32 lane-instructions per interaction (SURVEY 8(d)) x "
                            "interactions per launch / mean force-kernel time (CUDA events on the launching stream, live in this run); "
                            f"peak = 148 SM x 128 lanes x {sm_max:.0f} MHz ({peaks_src} max SM clock) x 2"),
                    "kernel_ms": f_us / 1e3,
                    "kernel_interactions_per_s": inter_per_launch / (f_us * 1e-6),
                    "flops47_tflops": FLOP47 * inter_per_launch / (f_us * 1e-6) / 1e12,
                    "frac_at_measured_clock": (ach_inst / (SM_COUNT * FP32_LANES_PER_SM * clocks["sm_mhz"] * 1e6)) if clocks.get("sm_mhz") else None,
                    "kernel_share_of_step": f_us * args.steps / (ms_total * 1e3) if world == 1 else None,
                    "measured_ceilings": ceilings,
                    "pipe_busy_equivalent": (FP32_INSTR_PER_INTERACTION + 3 * int(newton)) / FP32_INSTR_PER_INTERACTION * ach_inst / peak_inst,
                    "predictor_gbs": (n * (76 + 40)) / (float(np.mean(pred_us)) * 1e-6) / 1e9,
                    "hbm_peak_gbs": peaks.get("hbm_gbs")}
        out = {"metric": METRIC, "value": value, "unit": "interactions/s", "n_gpus": world, "steps": args.steps,
               "warmup": max(args.warmup, 3), "ms_per_step": ms_total / args.steps, "higher_is_better": True,
               "scaling": "strong", "vs_baseline": None, "dtype": "f32 (double-single separations, fp64 accumulation across tiles)",
               "data": "synthetic",
               "config": bench_config(inputs, n, eps2, int(newton), world),
               "gflops_60": value * FLOP_PAPER / 1e9, "gflops_66": value * 66 / 1e9,
               "clocks": clocks, "roofline": roofline, "gpu_launches": 4 * args.steps,
               "wall_s_timed_region": wall}
        if e2e:
            out["e2e"] = e2e
        if sweep is not None:
            out["ni_sweep"] = sweep
        if nb_cost is not None:
            out["neighbour_lists"] = nb_cost
        if ds_cost is not None:
            out["double_single_cost"] = ds_cost
        if c3 is not None:
            out["c3_sweep"] = c3
        if c2 is not None:
            out["c2_hermite"] = c2
        if not args.no_cpu_baseline and world == 1:
            rate, rows, dt, cores = cpu_oracle_rate(x, v, m, eps2, idx, args.cpu_seconds)
            out["cpu_baseline"] = {"value": rate, "unit": "interactions/s", "cores": cores, "kind": "oracle",
                                   "sample": f"{rows} randomly chosen i-rows x all {n} j of the same workload, {dt:.1f} s"}
        print(json.dumps(out), flush=True)

    g6.g6_close(0)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
