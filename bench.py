#!/usr/bin/env python
"""bench.py -- events/s of the summed squared helicity amplitude of u ubar -> n gamma on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4gamma] [--precision fp64]
                    [--impl ours|reference] [--no-sweep]

A step is one pass of the hot path over one batch of the named synthetic workload:
heget_amp2 (rows a1-a8 of DESIGN.md) followed by heget_xsec_reduce (a9-a10), inputs (momenta,
weights) resident in HBM.  `e2e` is the same through heget_xsec_host with pinned HOST buffers
(H2D and D2H copies inside the timed region).  One JSON line is printed by rank 0.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "events/s of summed |M|^2 for u ubar->n gamma"
# dram__bytes_read.sum + dram__bytes_write.sum of one amp2 launch at the config's full size, from
# the `ncu --set full` captures summarised under profiles/ (n, precision) -> bytes
NCU_DRAM_BYTES = {(4, "fp64"): 210208512, (4, "fp32"): 210454784, (8, "fp64"): 21140480, (8, "fp32"): 21051648}
# flop per event of amp2_kernel as ncu counts them over the whole kernel, tables included
# (smsp__sass_thread_inst_executed_op_{f,d}{fma x2, mul, add}_pred_on of the same captures / events)
NCU_FLOPS_PER_EVENT = {(4, "fp64"): 8815.0, (4, "fp32"): 7865.1, (8, "fp64"): 1.4349e8, (8, "fp32"): 1.4346e8}
UNIT = "events/s"


def model_flops_per_event(n):
    """Model C of DESIGN.md: permutation tree with prefix reuse, Weyl form, the 2*2^n non-zero
    helicity assignments; 44 flop per internal node, 24 per leaf (FMA = 2)."""
    internal = sum(math.factorial(n) // math.factorial(n - l) for l in range(1, n))
    return 2 * 2 ** n * (44 * internal + 24 * math.factorial(n))


def executed_flops_per_event(n, precision="fp32"):
    """What amp2_kernel executes: 2^n lanes (sigma_1 = +1 only, doubled by
    parity), tables excluded.
    n >= 5 (v9, factorised nodes psi = z v, csrc/amp2_chain.cuh): every ordered prefix of up to n-3
    photons is rho (4 FMA) + the vector v of the node (5 FMA + 1 MUL) + the accumulation rho A
    (4 FMA) = 27 flop, every prefix of n-2 photons (its two remaining orderings closed by the
    per-event table of closing dots) rho + accumulation = 16 flop.
    n = 4 (v8): one fvixx0 node = 16 FMA + 4 MUL = 36 flop for every ordered prefix of up to n-2
    photons and one dot product with the pair closing table, 8 FMA = 16 flop, per prefix of n-2
    photons; the first two tree levels once per event (48 entries psi_2 in factorised form, 42 flop
    each) instead of once per lane (16 nodes).  n = 2, 3 (v7): 36 flop per node and two vertex + closing-table dots,
    2 x (16 + 16) = 64 flop, per prefix of n-2 photons.  Cross-checked against ncu's
    sass_thread_inst_executed_op_{f,d}{fma,mul,add} counters in profiles/."""
    if n >= 5:
        upper = sum(math.factorial(n) // math.factorial(n - l) for l in range(1, n - 2))
        return 2 ** n * (27 * upper + 16 * (math.factorial(n) // 2))
    upper = sum(math.factorial(n) // math.factorial(n - l) for l in range(1, n - 1))
    closing = 16 if n >= 4 else 64
    flops = 2 ** n * (36 * upper + closing * (math.factorial(n) // 2))
    if n == 4:
        flops -= 2 ** n * 16 * 36 - 48 * 42   # 48 entries psi_2 = rho v per event, 42 flop each (factorised form)
    return flops


def _binom(n, k):
    return math.factorial(n) // (math.factorial(k) * math.factorial(n - k))


def executed_flops_per_event_algo(n, algo, precision="fp32"):
    """Executed flops of the separately named algorithms, tables excluded.
    subset: level m holds C(n,m) 2^m items of m vertex accumulations (8 FMA + 4 ADD = 20 flop) and
    one propagator (8 FMA + 4 MUL = 20 flop); 2^n closings of n terms (4 FMA + 2 ADD = 10 flop).
    two-sided: per lane the tree to depth n-KS-1 (36 flop per node) and n!/KS! closings of a vertex and a
    dot product (32 flop), plus the ubar-side table, C(n,m) 2^m entries of m x 40 flop for m = 2..KS and
    the folded last propagator (20 flop per entry of level KS), KS = min(n,4)."""
    if algo == "tree":
        return executed_flops_per_event(n, precision)
    if algo == "subset":
        return sum(_binom(n, m) * 2 ** m * (20 * m + 20) for m in range(1, n)) + 2 ** n * 10 * n
    ks = min(n, 4)
    closings = math.factorial(n) // math.factorial(ks)
    if ks == n:                                   # no u-side tree: one dot product per lane
        per_lane = 16 * closings
    else:                                         # full nodes above the last u-side photon, vertex + dot there
        nodes = sum(math.factorial(n) // math.factorial(n - l) for l in range(1, n - ks))
        per_lane = 36 * nodes + 32 * closings
    table = sum(_binom(n, m) * 2 ** m * m * 40 for m in range(2, ks + 1))
    if ks < n:
        table += _binom(n, ks) * 2 ** ks * 20     # last propagator folded into the table
    return 2 ** n * per_lane + table


ALGOS = {"tree": 0, "subset": 1, "two-sided": 2}
KERNEL_NAME = {"tree": "amp2_kernel", "subset": "amp2_subset_kernel", "two-sided": "amp2_twosided_kernel"}


def theoretical_peak(precision, sm_count, sm_max_mhz):
    lanes = 128 if precision == "fp32" else 64       # FP32 / FP64 FMA lanes per SM on B200
    return sm_count * lanes * 2 * sm_max_mhz * 1e6


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region: through NVML in-process
    (about a millisecond per sample, so even a 15 ms region gets several), else by polling
    nvidia-smi."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.index, self.sm, self.mx, self.reasons = index, [], [], set()
        self._stop, self._t, self.source = threading.Event(), None, "nvidia-smi"
        self._nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            phys = int(vis.split(",")[index]) if vis and vis.split(",")[index].isdigit() else index
            self._h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self._nvml, self.source = pynvml, "nvml"
        except Exception:
            self._nvml = None

    def _sample_nvml(self):
        n = self._nvml
        self.sm.append(float(n.nvmlDeviceGetClockInfo(self._h, n.NVML_CLOCK_SM)))
        self.mx.append(float(n.nvmlDeviceGetMaxClockInfo(self._h, n.NVML_CLOCK_SM)))
        get = getattr(n, "nvmlDeviceGetCurrentClocksEventReasons", None) or n.nvmlDeviceGetCurrentClocksThrottleReasons
        mask = int(get(self._h))
        bits = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40, "sw_power_cap": 0x4}
        for name, bit in bits.items():
            if mask & bit:
                self.reasons.add(name)

    def _sample_smi(self):
        out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                              "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout.strip()
        r = [x.strip() for x in out.split(",")] if out else []
        if len(r) >= 7:
            if r[0].replace(".", "").isdigit():
                self.sm.append(float(r[0]))
            if r[1].replace(".", "").isdigit():
                self.mx.append(float(r[1]))
            for i, name in enumerate(self.NAMES):
                if r[3 + i] == "Active":
                    self.reasons.add(name)

    def _run(self):
        while not self._stop.is_set():
            try:
                if self._nvml:
                    self._sample_nvml()
                else:
                    self._sample_smi()
            except Exception:
                pass
            self._stop.wait(0.002 if self._nvml else 0.1)

    def start(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()

    def stop(self):
        self._stop.set()
        if self._t:
            self._t.join(timeout=6)
        sm = sorted(self.sm)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(self.mx) if self.mx else None,
                "reasons": [n for n in self.NAMES if n in self.reasons], "samples": len(sm), "source": self.source}


def oracle_sample_events(cfg, seconds_budget=12.0):
    """How many events of this config the oracle is timed on: a BOUNDED sample sized for about
    `seconds_budget` seconds of wall time on this host (10-30 s of CPU work on all its cores),
    from a one-second pilot run of the oracle itself."""
    cores = os.cpu_count() or 1
    per_event_core_s = {2: 2e-6, 3: 2.5e-5, 4: 1e-4, 5: 1.5e-3, 6: 2.5e-2, 7: 0.4, 8: 6.0}[cfg["n"]]
    pilot = max(min(int(1.0 * cores / per_event_core_s), cfg["N"]), 1)
    rate, _, _ = time_oracle(cfg, pilot)
    want = int(rate * seconds_budget)
    # at least one event (the oracle spreads a single event's helicity assignments over the cores)
    return max(min(want, cfg["N"]), 1)


def time_oracle(cfg, n_events):
    """The oracle as it stands (oracle<double>, OpenMP over its own events) on the host cores."""
    import oracle
    from paper_0908_4403_b200 import workloads
    mom, _ = oracle.gen_events(cfg["seed"], cfg["n"], n_events, mode=cfg["mode"], a=cfg["a"], b=cfg["b"],
                               y_max=cfg["y_max"], apply_cuts=cfg["apply_cuts"], pt_cut=workloads.PT_CUT,
                               eta_cut=workloads.ETA_CUT, dr_cut=workloads.DR_CUT)
    t0 = time.perf_counter()
    oracle.amp2(mom)
    dt = time.perf_counter() - t0
    return n_events / dt, dt, oracle.num_threads()


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, same config/metric/unit."""
    from paper_0908_4403_b200 import workloads
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg = workloads.CONFIGS[args.config]
    n_ev = oracle_sample_events(cfg, seconds_budget=8.0)
    for _ in range(args.warmup):
        time_oracle(cfg, max(n_ev // 8, 1))
    total, cores = 0.0, 1
    for _ in range(args.steps):
        _, dt, cores = time_oracle(cfg, n_ev)
        total += dt
    value = n_ev * args.steps / total
    sample = "first %d of %d events of %s per step, oracle<double>, OpenMP" % (n_ev, cfg["N"], args.config)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.config, "n_photons": cfg["n"], "events_per_step": n_ev},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def time_config(hg, torch, name, precision, steps, warmup, flush, first_event, n_local, algo=0):
    """Device-timed steps of amp2 + xsec_reduce on resident inputs.  Returns per-step ms (whole
    step) and the amp2 kernel's own ms, both from CUDA events on the launching stream."""
    from paper_0908_4403_b200 import FP32, FP64, workloads
    cfg = workloads.CONFIGS[name]
    prec = FP64 if precision == "fp64" else FP32
    mom, w = hg.gen_events(cfg["seed"], cfg["n"], n_local, mode=cfg["mode"], a=cfg["a"], b=cfg["b"],
                           y_max=cfg["y_max"], apply_cuts=cfg["apply_cuts"], first_event=first_event)
    amp2 = torch.empty(n_local, dtype=torch.float64, device=hg.device)
    out3 = torch.empty(3, dtype=torch.float64, device=hg.device)

    def step(ev=None):
        if ev:
            ev[0].record()
        hg.amp2(mom, prec, out=amp2, algo=algo)
        if ev:
            ev[1].record()
        hg.xsec_reduce(amp2, w, cfg["n"], out3=out3)
        if ev:
            ev[2].record()

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
    return mom, w, out3, step, evs, flush


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="4gamma")
    ap.add_argument("--precision", default="fp64", choices=["fp32", "fp64"])
    ap.add_argument("--algo", default="tree", choices=sorted(ALGOS),
                    help="organisation of the permutation sum timed in the headline line (heget_amp2_algo); "
                         "tree = the north-star method and the default")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-sweep", action="store_true", help="skip the per-n / per-precision table")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    import torch.distributed as dist
    from paper_0908_4403_b200 import FP32, FP64, Heget, workloads

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    hg = Heget(local_rank, workloads.ALPHA, workloads.Q_U, workloads.PT_CUT, workloads.ETA_CUT, workloads.DR_CUT)
    cfg = workloads.CONFIGS[args.config]
    n = cfg["n"]
    # weak scaling: every rank processes the full per-GPU batch of the config, on its own
    # contiguous range of global event indices (no data-path collective; the three sums of
    # the reduction are all-reduced once per step)
    n_local = cfg["N"]
    first_event = rank * n_local
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=hg.device)   # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed_run(name, precision, steps, warmup, algo=0):
        c = workloads.CONFIGS[name]
        nl = c["N"]
        mom, w, out3, step, evs, _ = time_config(hg, torch, name, precision, steps, warmup, None, rank * nl, nl, algo)
        barrier()
        for ev in evs:
            flush_buf.zero_()                                  # L2 flush, outside the timed events
            step(ev)
            if world > 1:
                dist.all_reduce(out3)
        barrier()
        step_ms = [e[0].elapsed_time(e[2]) for e in evs]
        amp_ms = [e[0].elapsed_time(e[1]) for e in evs]
        return sum(step_ms), sum(amp_ms) / len(amp_ms), min(amp_ms), out3.cpu().numpy(), nl

    launches0 = hg.launch_count()
    sampler = ClockSampler(local_rank)
    sampler.start()
    total_ms, amp_ms, amp_ms_best, sums, nl = timed_run(args.config, args.precision, args.steps, args.warmup,
                                                         algo=ALGOS[args.algo])
    clocks = sampler.stop()
    launches = hg.launch_count() - launches0 - 3 * args.warmup - 1   # minus warm-up steps and the generator
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=hg.device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = t.item()
    value = world * nl * args.steps / (total_ms * 1e-3)

    # end to end through the host-buffer entry point (pinned host inputs, H2D + D2H inside)
    mom_d, w_d = hg.gen_events(cfg["seed"], n, nl, mode=cfg["mode"], a=cfg["a"], b=cfg["b"], y_max=cfg["y_max"],
                               apply_cuts=cfg["apply_cuts"], first_event=first_event)
    mom_h = torch.empty(mom_d.shape, dtype=torch.float64).pin_memory()
    w_h = torch.empty(w_d.shape, dtype=torch.float64).pin_memory()
    mom_h.copy_(mom_d)
    w_h.copy_(w_d)
    out3_h = torch.empty(3, dtype=torch.float64).pin_memory()
    prec = FP64 if args.precision == "fp64" else FP32
    for _ in range(2):
        hg.xsec_host(mom_h, w_h, prec, out3=out3_h)
    barrier()
    e2e_steps = max(1, min(args.steps, 5))
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        hg.xsec_host(mom_h, w_h, prec, out3=out3_h)
    barrier()
    e2e_s = time.perf_counter() - t0
    if world > 1:
        t = torch.tensor([e2e_s], dtype=torch.float64, device=hg.device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = t.item()
    e2e_value = world * nl * e2e_steps / e2e_s

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # roofline of the dominant kernel (amp2): plain-ALU bound.  `achieved` = flops the kernel
    # executes (the ncu-counted figure is the %peak figure) over its own time;
    # model C (the survey's algorithmic count, which ignores the parity relation and the
    # normalised E' entries) over the same time is given beside it as the cross-check.
    peak_measured = hg.fma_peak(prec, 0)
    peak_3reg = hg.fma_peak(prec, 1)
    peak_node = hg.fma_peak(prec, 2)
    sm_max = clocks["sm_max_mhz"] or 1965.0
    peak_theory = theoretical_peak(args.precision, torch.cuda.get_device_properties(local_rank).multi_processor_count, sm_max)
    tree_model = executed_flops_per_event_algo(n, args.algo, args.precision)
    counted = NCU_FLOPS_PER_EVENT.get((n, args.precision)) if args.algo == "tree" else None
    flops_per_event = counted if counted is not None else tree_model
    achieved = flops_per_event * nl / (amp_ms * 1e-3)
    model_c = model_flops_per_event(n) * nl / (amp_ms * 1e-3)
    roofline = {"bound": "alu", "achieved": achieved / 1e12, "peak": peak_measured / 1e12, "unit": "TFLOP/s",
                "frac": achieved / peak_measured, "traffic": NCU_DRAM_BYTES.get((n, args.precision)) if args.algo == "tree" else None,
                "kernel": "%s<%d,%s>" % (KERNEL_NAME[args.algo], n, "double" if prec == FP64 else "float"),
                "kernel_ms": amp_ms, "kernel_ms_best": amp_ms_best,
                "flops_per_event": flops_per_event,
                "flops_source": ("ncu-counted over the whole kernel, tables included (profiles/)" if counted is not None
                                 else "executed-instruction model of the tree, tables (< 1 % from 6 photons on) excluded"),
                "flops_per_event_executed": tree_model,
                "tree_model_tflops": tree_model * nl / (amp_ms * 1e-3) / 1e12,
                "peak_source": "heget_fma_peak on this GPU: FMA with constant-bank operands "
                               "(MEASURED_PEAKS.json has no non-tensor figure)",
                "peak_theoretical": peak_theory / 1e12, "frac_of_theoretical": achieved / peak_theory,
                "peak_three_register_fma": peak_3reg / 1e12, "peak_node_pattern": peak_node / 1e12,
                "frac_of_node_pattern": achieved / peak_node,
                "model_c_tflops": model_c / 1e12, "model_c_frac": model_c / peak_measured,
                "frac_note": "frac counts EXECUTED flops (what ncu counts); model_c_frac counts SURVEY 8(d)'s fixed "
                             "algorithmic figure (model C) over the same time.  Work removed by the parity relation and "
                             "by re-associating or sharing factors lowers frac while events/s and model_c_frac rise "
                             "(4 gamma fp64: v3 1.48 ms, frac 0.56 -> v7 1.02 ms, 0.48 -> v8 0.745 ms, 0.41 -> v9 0.70 ms, 0.39)",
                "flops_model": "executed: n = 4: 2^n lanes x (36 flop per tree node down to depth n-2 + 16 per pair of last "
                               "orderings, one dot with the pair closing table); n >= 5: 2^n lanes x (27 flop per factorised "
                               "node down to depth n-3 + 16 per node of n-2 photons), see executed_flops_per_event; model C (SURVEY 8(d)): 2*2^n x (44 per node "
                               "+ 24 per leaf), 3-5x the executed count because the kernel evaluates sigma_1=+1 only "
                               "(parity), uses normalised polarisation blocks and contracts the last two vertices and "
                               "the last propagator of both final orderings into a per-event table"}

    result = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
              "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
              "scaling": "weak", "vs_baseline": None, "dtype": "f64" if prec == FP64 else "f32",
              "data": "synthetic",
              "config": {"workload": args.config, "n_photons": n, "events_per_gpu": nl, "algo": args.algo,
                         "generation": "device Philox4x32-10 + RAMBO, seed %d" % cfg["seed"],
                         "l2": "256 MiB buffer written between timed steps (L2 flush)"},
              "clocks": clocks,
              "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(mom_h.numel() * 8 + w_h.numel() * 8),
                      "d2h_bytes_per_step": 24, "steps": e2e_steps},
              "gpu_launches": int(launches),
              "roofline": roofline,
              "xsec": {"sum_wA": float(sums[0]), "sum_wA2": float(sums[1]), "n_pass": float(sums[2])}}

    if not args.no_cpu_baseline:
        n_ev = oracle_sample_events(cfg)
        v, dt, cores = time_oracle(cfg, n_ev)
        result["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                  "sample": "first %d of %d events of %s, oracle<double>, %.1f s" % (n_ev, cfg["N"], args.config, dt)}

    if not args.no_sweep and world == 1:
        table = []
        for name in workloads.ORDER:
            for precision in ("fp32", "fp64"):
                _, a_ms, a_best, _, nn = timed_run(name, precision, 3, 3)
                nph = workloads.CONFIGS[name]["n"]
                pk = peak_measured if precision == args.precision else hg.fma_peak(FP64 if precision == "fp64" else FP32)
                ach = executed_flops_per_event(nph, precision) * nn / (a_ms * 1e-3)
                for algo_id, algo_name, note in (
                        (1, "subset", "HEGET_ALGO_SUBSET (heget_amp2_algo): not the permutation tree, own flop count"),
                        (2, "two-sided", "HEGET_ALGO_TREE2 (heget_amp2_algo): tree from u to depth n-4, closed with "
                                         "row vectors chained from ubar; own flop count")):
                    _, s_ms, _, _, _ = timed_run(name, precision, 3, 3, algo=algo_id)
                    s_fl = executed_flops_per_event_algo(nph, algo_name, precision) * nn / (s_ms * 1e-3)
                    table.append({"workload": name, "n": nph, "precision": precision, "events": nn, "algo": algo_name,
                                  "amp2_ms": s_ms, "events_per_s": nn / (s_ms * 1e-3),
                                  "executed_tflops": s_fl / 1e12, "frac_of_measured_peak": s_fl / pk, "note": note})
                table.append({"workload": name, "n": nph, "precision": precision, "events": nn, "algo": "tree",
                              "amp2_ms": a_ms, "events_per_s": nn / (a_ms * 1e-3),
                              "executed_tflops": ach / 1e12, "frac_of_measured_peak": ach / pk,
                              "model_c_tflops": model_flops_per_event(nph) * nn / (a_ms * 1e-3) / 1e12})
        result["per_config"] = table

    if not args.no_sweep and world == 1:
        # NEXT-1 entry points on the headline workload: one drawn helicity per event, Fig. 2 histogram
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        val, _ = hg.amp2_sampled(cfg["seed"], mom_d, prec)
        hg.histogram(mom_d, val, 0, 0.0, 1500.0, 60)
        torch.cuda.synchronize()
        ev[0].record()
        val, _ = hg.amp2_sampled(cfg["seed"], mom_d, prec)
        ev[1].record()
        hg.histogram(mom_d, val, 0, 0.0, 1500.0, 60)
        ev[2].record()
        torch.cuda.synchronize()
        ev2 = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        hg.list2(cfg["seed"], mom_d, prec)
        torch.cuda.synchronize()
        ev2[0].record()
        hg.list2(cfg["seed"], mom_d, prec)
        ev2[1].record()
        torch.cuda.synchronize()
        # the paper's arithmetic for the headline quantity on this GPU: List 2 called for all 4*2^n
        # helicity assignments per thread (model A of SURVEY 8(d)); bounded to n <= 6
        if n <= 6:
            n_pd = nl if n <= 4 else nl // 64
            ev3 = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
            sub = mom_d[:n_pd].contiguous()
            hg.list2_sum(sub, prec)
            torch.cuda.synchronize()
            ev3[0].record()
            hg.list2_sum(sub, prec)
            ev3[1].record()
            torch.cuda.synchronize()
            pd_ms = ev3[0].elapsed_time(ev3[1])
            result["paper_design"] = {"events_per_s": n_pd / (pd_ms * 1e-3), "ms": pd_ms, "events": n_pd,
                                      "note": "heget_list2_sum: the paper's List 2 program (thread per event, "
                                              "4-component, no prefix reuse, no parity) looped over all helicity "
                                              "assignments, same GPU, same precision, same momenta"}
        result["next1"] = {"paper_list2_ms": ev2[0].elapsed_time(ev2[1]),
                           "paper_list2_events_per_s": nl / (ev2[0].elapsed_time(ev2[1]) * 1e-3),
                           "paper_list2_note": "heget_list2: the paper's List 2 program (thread per event, 4-component, "
                                               "no reuse) on this GPU, same estimator as amp2_sampled",
                           "amp2_sampled_ms": ev[0].elapsed_time(ev[1]),
                           "amp2_sampled_events_per_s": nl / (ev[0].elapsed_time(ev[1]) * 1e-3),
                           "histogram_ms": ev[1].elapsed_time(ev[2]), "events": nl, "precision": args.precision}

    print(json.dumps(result))
    hg.close()


if __name__ == "__main__":
    main()
