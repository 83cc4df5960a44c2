#!/usr/bin/env python
"""bench.py -- chi0 pair transitions/s and rank-K FP64 TFLOP/s on BASELINE.json configs[1] (molecule-in-box).

A step is one pass of the whole hot path over the workload (S1 = create is done
once, untimed): reset, rpa_chi0_add_kpoint for every k-point of the rank, rpa_chi0_get for every omega and
rpa_ec_q.  `value` = transitions of all ranks / max-over-ranks device time, inputs resident in HBM.
`e2e` = the same pass in the paper's data flow: plane-wave coefficients and projections start in pinned HOST memory,
are copied and expanded on the device (Eq. 10) inside the timed region, and E_c(q) / e(omega) are read back to the
host; `e2e_grid` = the same with grid orbitals uploaded instead (20x the bytes, PCIe-bound).  Everything is FP64 / complex128; `roofline` is the FP64
tensor-core rank-K kernel (rank_k3m_kernel) in TFLOP/s.  Extra blocks of the same JSON line: `rank_k_i8` (the
opt-in int8-sliced arm, timed in the same run and compared with the FP64 result), `per_config` (configs 0 and 2
in full, configs 3 and 4 on one 8192-transition batch at full grid / nG), `cpu_baseline` (the oracle).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--impl reference]
    torchrun --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P bench.py --gpus N ...

N > 1: weak scaling, no data-path collective -- every rank owns one k-point of an N-k-point problem (P:L181:
"no MPI communication throughout steps 2-11"); the one exchange of the method, the sum of the per-rank
accumulators at the end of a q, is an NCCL all-reduce inside the timed step.
"""
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

from paper_1307_8052_b200 import workload as W  # noqa: E402

METRIC = "chi0 pair transitions/s (rank-K FP64 TFLOP/s in roofline), 1 q-point, all omega"
UNIT = "transitions/s"
MIN_WARMUP = 3   # timing rule of the bench contract: at least 3 untimed steps
# dram__bytes_read.sum + dram__bytes_write.sum of rank_k3m_kernel from the ncu --set full capture named beside it: one
# batch of configs[1] (7200 transitions x 16 omega) = its whole-wave launch + its K-sliced tail launch.  A constant
# copied from that profile, NOT measured in the run that prints it: `traffic_from` says so in the JSON.
RANK_K_DRAM_TRAFFIC = {1: (2188.7e6, "profiles/r2h_rank_k3m.md")}
RANK_K_I8_DRAM_TRAFFIC = {1: (4455.9e6, "profiles/r1i_bench_cfg1.md")}


def rank_k_useful_flops(ng, n_omega, n_pairs):
    """8 flop per complex MAC on one triangle: 4 nG (nG+1) n_omega per pair."""
    return 4.0 * ng * (ng + 1) * n_omega * n_pairs


class ClockSampler:
    """nvidia-smi clocks + throttle reasons every 50 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); power.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            return json.load(fh), "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0}, "fallback (B200_PROFILING.md)"


def config_dict(cfg, ng, world, batch, exchange):
    """The `config` object of the JSON line -- the same for our arm and for --impl reference."""
    return {"workload": f"configs[{cfg.index}] {cfg.name}", "grid": list(cfg.grid), "n_k_per_gpu": cfg.n_k,
            "n_occ": cfg.n_occ, "n_unocc": cfg.n_unocc, "n_pairs": cfg.n_pairs * world, "nG": int(ng), "n_omega": cfg.n_omega,
            "atoms_x_proj": [cfg.n_atoms, cfg.n_proj_per_atom], "max_batch_pairs": batch or 8192,
            "l2": "inputs (%.2f GB of orbitals per k-point) exceed the 126 MB L2; no explicit flush" %
                  ((cfg.n_occ + cfg.n_unocc) * cfg.n_grid * 16 / 1e9),
            "step": "reset + add_kpoint (S2-S6) + get x n_omega (S7) + ec_q (S8)",
            "parallelism": "1 GPU" if world == 1 else f"k-points sharded over {world} GPUs + {exchange} of S"}


# ------------------------------------------------------------------------------------------------ reference arm
def oracle_sample(cfg, budget_s, chunk=64, with_ec=True):
    """The oracle, as it stands, on a bounded sample of the workload: slices of `chunk` unoccupied bands against
    one occupied band of k-point 0 (full grid / nG / omega / atoms) are added until `budget_s` seconds of CPU
    work are spent, then (with_ec) E_c(q) is taken on the full nG x nG matrices.  Returns
    (pairs, t_add, t_ec, estimated whole-workload transitions/s, threads, nG)."""
    import oracle
    om, wt = W.omega_grid(cfg.n_omega)
    orc = oracle.Chi0Oracle(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt)
    Q, R = W.paw_Q(cfg, orc.K2), W.atom_positions(cfg)
    pairs, t_add, n, m0 = 0, 0.0, 0, 0
    while t_add < budget_s and n < cfg.n_occ:
        m1 = min(m0 + chunk, cfg.n_unocc)
        kd = W.kpoint(cfg, 0, occ=[n], unocc=range(m0, m1))
        t0 = time.perf_counter()
        orc.add_kpoint(kd, cfg.n_proj, Q, R)
        t_add += time.perf_counter() - t0
        pairs += m1 - m0
        m0 = m1
        if m0 >= cfg.n_unocc:
            n, m0 = n + 1, 0
    t_ec = 0.0
    if with_ec:
        t1 = time.perf_counter()
        orc.ec_q(W.coulomb(orc.K2))
        t_ec = time.perf_counter() - t1
    est = cfg.n_pairs / (cfg.n_pairs * t_add / pairs + t_ec)
    return pairs, t_add, t_ec, est, oracle.num_threads(), orc.ng


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    world = int(os.environ.get("WORLD_SIZE", "1"))
    budget = min(args.ref_seconds, 150.0 / max(1, args.warmup + args.steps))
    vals, ts = [], []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        pairs, t_add, t_ec, est, cores, ng = oracle_sample(cfg, budget)
        if i >= args.warmup:
            vals.append(est)
            ts.append(time.perf_counter() - t0)
    v = float(np.mean(vals))
    sample = (f"per step: {pairs} transitions of k-point 0 (64-band slices, full grid/nG/omega/atoms, {budget:.0f} s "
              f"budget) + E_c(q) on the full nG x nG matrices; value = n_pairs / (n_pairs * t_add/pairs_sampled + t_ec)")
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(ts)), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64 (complex128)", "data": "synthetic",
            "config": config_dict(cfg, ng, world, args.batch, args.exchange),
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------------ our arm
def stage_report(B, cfg, ng, pairs_per_step, steps, stage_ms, stage_n, peak_tf, peaks, peak_kind):
    """Per-stage rooflines from the library's own CUDA events (rpa_chi0_stage_times) over `steps` timed steps."""
    rk_launches = int(stage_n[4])
    rk_ms = float(stage_ms[4]) / max(rk_launches, 1)
    rk_flops = rank_k_useful_flops(ng, cfg.n_omega, pairs_per_step * steps) / max(rk_launches, 1)
    rk_tf = rk_flops / (rk_ms * 1e-3) * 1e-12 if rk_ms > 0 else 0.0
    pd_ms = float(stage_ms[0] + stage_ms[1]) / steps
    pd_bytes = pairs_per_step * 16.0 * (cfg.n_grid + ng)   # 16 N per pair (stream psi_m) + 16 nG (write n)
    pd_gbs = pd_bytes / (pd_ms * 1e-3) * 1e-9 if pd_ms > 0 else 0.0
    return {"rank_k": {"tflops": rk_tf, "frac": rk_tf / peak_tf if peak_tf else None, "ms_per_launch": rk_ms,
                       "launches": rk_launches, "flops_per_launch": rk_flops, "ms_per_step": float(stage_ms[4]) / steps},
            "pair_density": {"bound": "hbm", "achieved": pd_gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                             "frac": pd_gbs / peaks["hbm_gbs"], "peak_kind": peak_kind, "ms_per_step": pd_ms,
                             "bytes_per_pair": 16.0 * (cfg.n_grid + ng)},
            "ms_per_step": {n: float(t) / steps for n, t in zip(B.STAGE_NAMES[:5], stage_ms[:5])},
            # stage 5 (rank_k_i8_mma) is a SUBSET of stage 4: it is not part of the sum
            "sum_ms": float(np.sum(stage_ms[:5])) / steps}


def run_ours(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_1307_8052_b200 import binding as B
    from paper_1307_8052_b200 import probes
    from paper_1307_8052_b200 import sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    warmup = max(args.warmup, MIN_WARMUP)

    om, wt = W.omega_grid(cfg.n_omega)
    ptot = int(cfg.n_proj.sum())
    h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, args.batch, ptot, dev)
    g, K2 = B.rpa_chi0_gvectors(h)
    ng = len(g)
    Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to(dev)
    R, npj = W.atom_positions(cfg), cfg.n_proj
    v = W.coulomb(K2)
    # weak scaling: this rank's k-points of a (world * n_k)-k-point problem; throughput does not depend on values
    my_k = [rank * cfg.n_k + k for k in range(cfg.n_k)]
    n_k_total = world * cfg.n_k
    t0 = time.perf_counter()
    # one generated k-point per rank is reused for all its k labels when n_k > 1 (no data-dependent
    # branching); configs[1] has a single k-point, so nothing is reused there
    kd = W.kpoint(cfg, my_k[0] % max(cfg.n_k, 1))
    gen_s = time.perf_counter() - t0
    host = {k: torch.from_numpy(getattr(kd, k)).pin_memory() for k in ("psi_occ", "psi_unocc", "P_occ", "P_unocc")}
    devt = {k: t.to(dev) for k, t in host.items()}
    kweight = 1.0 / n_k_total
    out = torch.empty((ng, ng), dtype=torch.complex128, device=dev)
    S = B.rpa_chi0_accumulators(h) if world > 1 else None

    g_pw, C_occ, C_unocc = W.kpoint_coefficients(cfg, kd.k)
    host_pw = {"C_occ": torch.from_numpy(C_occ).pin_memory(), "C_unocc": torch.from_numpy(C_unocc).pin_memory()}

    def step(from_host, tail_ms=None):
        B.rpa_chi0_reset(h)
        nb = 0
        for _ in my_k:
            if from_host == "pw":   # the paper's pipeline: coefficients up, Table 1 step 3 (Eq. 10) on the device
                nb += B.add_kpoint_host_pw(h, kweight, g_pw, host_pw["C_occ"], host_pw["C_unocc"], kd.eps_occ, kd.eps_unocc,
                                           kd.f_occ, kd.f_unocc, npj, host["P_occ"], host["P_unocc"], Qd, R)
            elif from_host:
                nb += B.add_kpoint_host(h, kd, npj, Qd, R, pinned=host, kweight=kweight)
            else:
                B.rpa_chi0_add_kpoint(h, kweight, devt["psi_occ"], devt["psi_unocc"], kd.eps_occ, kd.eps_unocc, kd.f_occ,
                                      kd.f_unocc, npj, devt["P_occ"], devt["P_unocc"], Qd, R)
        lo, hi = 0, cfg.n_omega
        if world > 1 and args.exchange == "reduce_scatter":
            lo, hi = sharding.reduce_scatter_accumulators(S, cfg.n_omega)   # this rank now owns frequencies [lo, hi)
        elif world > 1:
            sharding.allreduce_accumulators(S)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)] if tail_ms is not None else None
        if ev:
            ev[0].record()
        for i in range(lo, hi):
            B.rpa_chi0_get(h, i, out)
        if ev:
            ev[1].record()
        if (lo, hi) == (0, cfg.n_omega):
            ec, e = B.rpa_ec_q(h, v)  # blocks; reads E_c(q), e(omega) back to the host
        else:
            ec_part, e = B.rpa_ec_q_range(h, v, lo, hi)
            ec = sharding.allreduce_scalar(ec_part, dev)
        if ev:
            ev[2].record()
            ev[2].synchronize()
            tail_ms[0] += ev[0].elapsed_time(ev[1])
            tail_ms[1] += ev[1].elapsed_time(ev[2])
        return nb, ec, e

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(from_host, steps, n_warm, tail_ms=None):
        for _ in range(n_warm):
            step(from_host)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        nb = 0
        for _ in range(steps):
            nb, ec, e = step(from_host, tail_ms)
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        if world > 1:
            t = torch.tensor([ms], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        return ms / steps, nb, ec

    peak_tf = probes.rpa_probe_fp64_tensor_peak(dev)
    pairs_per_rank = len(my_k) * cfg.n_occ * cfg.n_unocc
    pairs_total = pairs_per_rank * world

    # ---- the headline: device-resident inputs, FP64 tensor-core rank-K (the library's default), clocks sampled ----------
    B.rpa_chi0_set_profiling(h, True)
    sampler = ClockSampler(local)
    for _ in range(warmup):
        step(False)
    barrier()
    B.rpa_chi0_set_profiling(h, True)  # zero the stage timers after warm-up
    launches0 = B.rpa_chi0_launch_count(h)
    if rank == 0:
        sampler.start()
    tail_ms = [0.0, 0.0]   # rpa_chi0_get x n_omega, rpa_ec_q (CUDA events on the handle's stream, inside the timed steps)
    ms_step, _, ec_dev = timed(False, args.steps, 0, tail_ms)
    clocks = sampler.stop() if rank == 0 else None
    launches = B.rpa_chi0_launch_count(h) - launches0
    stage_ms, stage_n = B.rpa_chi0_stage_times(h)
    B.rpa_chi0_set_profiling(h, False)
    fp_b, i8_b = B.rpa_chi0_rank_k_batches(h)
    assert i8_b == 0, "the headline must run the FP64 tensor kernel"
    chi_fp64 = [B.rpa_chi0_get(h, i).clone() for i in (0, cfg.n_omega // 2, cfg.n_omega - 1)]

    # end to end from pinned host memory
    ms_e2e, h2d, ec_e2e = timed(True, args.steps, max(1, warmup // 2))
    assert abs(ec_e2e - ec_dev) <= 1e-12 * abs(ec_dev), (ec_e2e, ec_dev)
    # end to end from the plane-wave coefficients in pinned host memory (orbitals expanded on the device)
    ms_pw, h2d_pw, ec_pw = timed("pw", args.steps, max(1, warmup // 2))
    assert abs(ec_pw - ec_dev) <= 1e-10 * abs(ec_dev), (ec_pw, ec_dev)

    # ---- extra arm: the opt-in int8-sliced rank-K (rpa_chi0_set_rank_k_mode), same handle, same inputs, same steps --------
    i8_arm = None
    if world == 1 and not args.no_i8_arm:
        digits = 7
        B.rpa_chi0_set_rank_k_mode(h, B.RPA_RANK_K_I8, digits)
        for _ in range(2):
            step(False)
        barrier()
        B.rpa_chi0_set_profiling(h, True)
        ms_i8, _, ec_i8 = timed(False, args.steps, 0)
        sm_i8, sn_i8 = B.rpa_chi0_stage_times(h)
        B.rpa_chi0_set_profiling(h, False)
        took_i8 = B.rpa_chi0_rank_k_batches(h)[1] > 0
        rel = [float((torch.linalg.norm(B.rpa_chi0_get(h, i) - ref) / torch.linalg.norm(ref)).item())
               for i, ref in zip((0, cfg.n_omega // 2, cfg.n_omega - 1), chi_fp64)]
        B.rpa_chi0_set_rank_k_mode(h, B.RPA_RANK_K_FP64_3M, 0)
        if took_i8 and int(sn_i8[5]) > 0:
            i8_peak, i8_bad = probes.rpa_probe_int8_tensor_peak(dev)
            n5 = int(sn_i8[5])
            mma_ms = float(sm_i8[5]) / n5
            # int8 operations the emulation issues: digit pairs i + j < digits, both halves (Re, Im) of the lower triangle, K' = 2K
            ops = (digits * (digits + 1) // 2) * 2.0 * cfg.n_omega * ng * (ng + 1) * 2.0 * pairs_per_rank * args.steps / n5
            tops = ops / (mma_ms * 1e-3) * 1e-12
            stage_i8 = float(sm_i8[4]) / args.steps
            peaks_, _ = measured_peaks()
            i8_arm = {"mode": "rpa_chi0_set_rank_k_mode(RPA_RANK_K_I8, digits) -- opt-in, NOT the library default",
                      "digits": digits, "ms_per_step": ms_i8, "rank_k_stage_ms_per_step": stage_i8,
                      "mma_ms_per_launch": mma_ms, "mma_launches": n5, "int8_tops": tops, "int8_peak_probe_tops": i8_peak,
                      "frac": tops / i8_peak if i8_peak else None,
                      "int8_peak_from_bf16_tops": peaks_.get("bf16_tflops", 0) * 4.5 / 2.25,
                      "frac_vs_bf16_scaled_peak": tops / (peaks_.get("bf16_tflops", 0) * 2.0) if peaks_.get("bf16_tflops") else None,
                      "probe_self_check_mismatches": i8_bad,
                      "fp64_equivalent_tflops": rank_k_useful_flops(ng, cfg.n_omega, pairs_per_rank) / (stage_i8 * 1e-3) * 1e-12,
                      "rel_fro_vs_fp64": max(rel), "ec_q_rel_diff_vs_fp64": abs(ec_i8 - ec_dev) / abs(ec_dev),
                      "traffic": RANK_K_I8_DRAM_TRAFFIC.get(cfg.index, (None, None))[0],
                      "traffic_from": RANK_K_I8_DRAM_TRAFFIC.get(cfg.index, (None, None))[1],
                      "note": "digit slices of the FP64 operands on the int8 tensor pipe (tcgen05), exact s32 products, FP64 "
                              "recombination; error bound per element in include/rpa_chi0.h; int8_tops counts the emulation's "
                              "own operations (28 digit pairs), not the method's flops"}
        else:
            i8_arm = {"mode": "RPA_RANK_K_I8", "note": "batches below the int8 thresholds: the FP64 kernel ran", "ms_per_step": ms_i8}

    if rank == 0:
        peaks, peak_kind = measured_peaks()
        rep = stage_report(B, cfg, ng, pairs_per_rank, args.steps, stage_ms, stage_n, peak_tf, peaks, peak_kind)
        rk = rep["rank_k"]
        traffic, traffic_from = RANK_K_DRAM_TRAFFIC.get(cfg.index, (None, None))
        peak_alt = peaks.get("bf16_tflops", 0) * 40.0 / 2250.0
        roofline = {"kernel": "rank_k3m_kernel", "bound": "tensor", "achieved": rk["tflops"], "peak": peak_tf, "unit": "TFLOP/s",
                    "frac": rk["frac"], "traffic": traffic, "traffic_from": traffic_from,
                    "peak_source": "FP64 DMMA issue rate measured live by librpa_probes.so rpa_probe_fp64_tensor_peak "
                                   "(register-only mma.sync.m8n8k4.f64, all SMs); MEASURED_PEAKS.json has no FP64 entry",
                    "peak_alt_tflops_from_bf16": peak_alt, "frac_vs_peak_alt": rk["tflops"] / peak_alt if peak_alt else None,
                    "note": "achieved = ALGORITHMIC flops (SURVEY 8(d): 4 nG (nG+1) n_omega per pair = 8 per complex "
                            "multiply-add on one triangle) / time; the kernel forms the complex product with 3 real "
                            "multiplications (3M), so it EXECUTES 3/4 of them on the tensor pipe: executed_frac = flops "
                            "actually issued / peak; one 'launch' here is the rank-K of one batch of transitions = its "
                            "whole-wave launch + the K-sliced launch of the last partial wave",
                    "executed_frac": 0.75 * rk["tflops"] / peak_tf if peak_tf else None,
                    "flops_per_launch": rk["flops_per_launch"], "ms_per_launch": rk["ms_per_launch"], "launches": rk["launches"],
                    "share_of_step": rk["ms_per_step"] / ms_step}
        line = {
            "metric": METRIC, "value": pairs_total / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64 (complex128)", "data": "synthetic",
            "config": config_dict(cfg, ng, world, args.batch, args.exchange),
            "clocks": clocks,
            # end to end in the paper's own data flow (Table 1 steps 3 and 5-13): the host holds the orbitals as
            # plane-wave coefficients; every step copies them (and the projections) from pinned host memory, expands them on
            # the device with rpa_pw_to_grid (Eq. 10, inside the timed region), adds the k-point, reads chi0 out for every
            # omega and reads E_c(q), e(omega) back to the host
            "e2e": {"value": pairs_total / (ms_pw * 1e-3), "unit": UNIT, "ms_per_step": ms_pw,
                    "h2d_bytes_per_step": int(h2d_pw), "d2h_bytes_per_step": 8 * (1 + cfg.n_omega) + 16,
                    "input": "plane-wave coefficients C_n(Q) + PAW projections in pinned host memory -> "
                             "binding.add_kpoint_host_pw (rpa_pw_to_grid + rpa_chi0_add_kpoint) -> rpa_chi0_get x n_omega -> rpa_ec_q"},
            # the same step when the caller holds the orbitals on the real-space grid in host memory (20x the bytes): the
            # upload of 2.1 GB per k-point at PCIe speed bounds it, whatever the kernels do
            "e2e_grid": {"value": pairs_total / (ms_e2e * 1e-3), "unit": UNIT, "ms_per_step": ms_e2e,
                         "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": 8 * (1 + cfg.n_omega) + 16,
                         "input": "grid orbitals u(r) in pinned host memory -> binding.add_kpoint_host (sliced, pipelined upload)"},
            "gpu_launches": int(launches),
            "roofline": roofline,
            "stages": {"ms_per_step": rep["ms_per_step"], "get_all_omega_ms": tail_ms[0] / args.steps,
                       "ec_q_ms": tail_ms[1] / args.steps, "sum_ms": rep["sum_ms"], "pair_density": rep["pair_density"]},
            "ec_q_ha": ec_dev, "gen_s": gen_s,
        }
        if args.warmup != warmup:
            line["warmup_requested"] = args.warmup
        if i8_arm is not None:
            line["rank_k_i8"] = i8_arm
    h.close()
    del devt, host, out, chi_fp64, Qd
    torch.cuda.empty_cache()
    if rank == 0:
        if world == 1 and not args.no_per_config:
            line["per_config"] = per_config_block(args, dev, peak_tf, peaks, peak_kind, line, cfg)
        if world == 1 and not args.no_cpu_baseline:
            pairs, t_add, t_ec, est, cores, _ = oracle_sample(cfg, args.ref_seconds)
            line["cpu_baseline"] = {"value": est, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"{pairs} transitions of k-point 0 (64-band slices, full grid/nG/omega/"
                                              f"atoms; {t_add:.1f} s) + E_c(q) on the full matrices ({t_ec:.1f} s); "
                                              f"value = n_pairs / (n_pairs * t_add/{pairs} + t_ec)"}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ---------------------------------------------------------------------------------------------- the other configs
PER_CONFIG_PLAN = {
    # index: (occupied bands, unoccupied bands) of the timed k-point; None = all of them
    0: (None, None),
    2: (None, None),
    3: (8, 1024),    # one batch of 8192 transitions at full grid / nG / omega / atoms
    4: (8, 1024),
}


def per_config_block(args, dev, peak_tf, peaks, peak_kind, main_line, main_cfg):
    """Driver-visible numbers for every BASELINE.json config (north_star: 'on all 5 configs').  Configs 0 and 2 run in
    full (config 2: one generated k-point reused for its 64 labels -- throughput does not depend on values); configs 3
    and 4 run ONE default-size batch of 8 x 1024 = 8192 transitions at full grid / nG / omega / atoms (their full steps
    take 3 s and 2 min).  Orbitals are expanded on the device from seeded plane-wave coefficients (rpa_pw_to_grid, outside
    the timed region).  Same step as the headline: reset + add_kpoint + get x n_omega + ec_q, device-resident inputs,
    FP64 tensor-core rank-K, CUDA events."""
    import torch
    from paper_1307_8052_b200 import binding as B
    out = {}
    steps, n_warm = 3, 2
    for idx, (n_o, n_u) in PER_CONFIG_PLAN.items():
        if idx == main_cfg.index:
            continue
        cfg = W.CONFIGS[idx]
        t_wall = time.perf_counter()
        om, wt = W.omega_grid(cfg.n_omega)
        ptot = int(cfg.n_proj.sum())
        h = B.rpa_chi0_create(cfg.grid, cfg.cell, cfg.q_red, W.tuned_ecut(cfg), om, wt, 0, ptot, dev)
        try:
            g, K2 = B.rpa_chi0_gvectors(h)
            ng = len(g)
            occ = list(range(cfg.n_occ if n_o is None else n_o))
            unocc = list(range(cfg.n_unocc if n_u is None else n_u))
            g_pw, C_o, C_u = W.kpoint_coefficients(cfg, 0, occ, unocc)
            psi_o = B.rpa_pw_to_grid(h, g_pw, torch.from_numpy(C_o).to(dev))
            psi_u = B.rpa_pw_to_grid(h, g_pw, torch.from_numpy(C_u).to(dev))
            eps, f = W.eigenvalues(cfg, 0)
            P = W.projections(cfg, 0)
            bo, bu = np.asarray(occ), np.asarray(unocc) + cfg.n_occ
            c = np.ascontiguousarray
            P_o, P_u = torch.from_numpy(c(P[bo])).to(dev), torch.from_numpy(c(P[bu])).to(dev)
            Qd = torch.from_numpy(W.paw_Q(cfg, K2)).to(dev)
            R, v = W.atom_positions(cfg), W.coulomb(K2)
            n_k = cfg.n_k if n_o is None else 1
            kw = 1.0 / cfg.n_k
            chi = torch.empty((ng, ng), dtype=torch.complex128, device=dev)
            tail = [0.0]

            def step(timed_tail=False):
                B.rpa_chi0_reset(h)
                for _ in range(n_k):
                    B.rpa_chi0_add_kpoint(h, kw, psi_o, psi_u, c(eps[bo]), c(eps[bu]), c(f[bo]), c(f[bu]), cfg.n_proj, P_o, P_u, Qd, R)
                for i in range(cfg.n_omega):
                    B.rpa_chi0_get(h, i, chi)
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record()
                ec, _ = B.rpa_ec_q(h, v)
                e1.record(); e1.synchronize()
                if timed_tail:
                    tail[0] += e0.elapsed_time(e1)
                return ec

            for _ in range(n_warm):
                step()
            torch.cuda.synchronize()
            B.rpa_chi0_set_profiling(h, True)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(steps):
                ec = step(True)
            b.record(); b.synchronize()
            ms = a.elapsed_time(b) / steps
            sm, sn = B.rpa_chi0_stage_times(h)
            B.rpa_chi0_set_profiling(h, False)
            pairs = n_k * len(occ) * len(unocc)
            rep = stage_report(B, cfg, ng, pairs, steps, sm, sn, peak_tf, peaks, peak_kind)
            entry = {"workload": f"configs[{idx}] {cfg.name}" + ("" if n_o is None else f": one batch of {len(occ)} x {len(unocc)} bands of k-point 0"),
                     "full_config": n_o is None, "grid": list(cfg.grid), "nG": ng, "n_pairs_timed": pairs, "ms": ms,
                     "transitions_per_s": pairs / (ms * 1e-3),
                     "rank_k_tflops": rep["rank_k"]["tflops"], "rank_k_frac": rep["rank_k"]["frac"],
                     "rank_k_ms": rep["rank_k"]["ms_per_step"],
                     "pair_density_gbs": rep["pair_density"]["achieved"], "pair_density_frac": rep["pair_density"]["frac"],
                     "pair_density_ms": rep["pair_density"]["ms_per_step"], "stage_ms": rep["ms_per_step"],
                     "paw_ms": rep["ms_per_step"]["paw"], "ec_q_ms": tail[0] / steps, "ec_q_ha": ec}
            if idx == 0:
                entry["note"] = "launch/latency-bound (8.7e7 flop in total): throughput only, no roofline claim"
        finally:
            h.close()
        del psi_o, psi_u, chi, Qd, P_o, P_u
        torch.cuda.empty_cache()
        if not args.no_cpu_baseline:
            # the oracle's accumulation rate on the same config (per-pair cost does not depend on the slice); E_c(q) left
            # out (unblocked Cholesky of 16 matrices of 5001: minutes)
            pairs_o, t_add, _, _, cores, _ = oracle_sample(cfg, 3.0, chunk=64 if idx in (0, 2) else 8, with_ec=False)
            entry["oracle_transitions_per_s"] = pairs_o / t_add
            entry["oracle_sample"] = f"{pairs_o} transitions, {t_add:.1f} s, {cores} threads, add_kpoint only"
        entry["wall_s"] = time.perf_counter() - t_wall
        out[str(idx)] = entry
    # the headline config in the same shape, from the main measurement
    st = main_line["stages"]
    out[str(main_cfg.index)] = {"workload": main_line["config"]["workload"], "full_config": True, "grid": list(main_cfg.grid),
                                "nG": main_line["config"]["nG"], "n_pairs_timed": main_line["config"]["n_pairs"],
                                "ms": main_line["ms_per_step"], "transitions_per_s": main_line["value"],
                                "rank_k_tflops": main_line["roofline"]["achieved"], "rank_k_frac": main_line["roofline"]["frac"],
                                "rank_k_ms": st["ms_per_step"]["rank_k"],
                                "pair_density_gbs": st["pair_density"]["achieved"], "pair_density_frac": st["pair_density"]["frac"],
                                "pair_density_ms": st["pair_density"]["ms_per_step"], "paw_ms": st["ms_per_step"]["paw"],
                                "ec_q_ms": st["ec_q_ms"], "ec_q_ha": main_line["ec_q_ha"]}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="index into BASELINE.json configs (default: 1, molecule)")
    ap.add_argument("--batch", type=int, default=0, help="max_batch_pairs (0: library default)")
    ap.add_argument("--ref-seconds", type=float, default=12.0, help="CPU seconds of oracle work per sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config block (configs 0, 2, 3, 4)")
    ap.add_argument("--no-i8-arm", action="store_true", help="skip the opt-in int8-sliced rank-K arm")
    ap.add_argument("--exchange", default="allreduce", choices=["allreduce", "reduce_scatter"],
                    help="N > 1: all-reduce of S (every rank reads out and factorises all frequencies) or reduce-scatter "
                         "by frequency (every rank reads out and factorises its own, scalar all-reduce of E_c)")
    ap.add_argument("--bands", default="", help="OxU: time only the first O occupied and U unoccupied bands per k-point "
                                                "(profiling runs of the big configs; named in config.workload)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    cfg = W.CONFIGS[args.config]
    if args.bands:
        import dataclasses
        n_o, n_u = (int(x) for x in args.bands.lower().split("x"))
        cfg = dataclasses.replace(cfg, n_occ=n_o, n_unocc=n_u, name=f"{cfg.name} (band slice {n_o} x {n_u})")
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
