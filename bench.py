#!/usr/bin/env python
"""bench.py -- events/s of the summed squared helicity amplitude of u ubar -> n gamma on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4gamma] [--precision fp64]
                    [--impl ours|reference] [--no-sweep] [--no-cpu-baseline]

A step is one pass of the hot path over one batch of the named synthetic workload:
heget_amp2 (rows a1-a8 of DESIGN.md) followed by heget_xsec_reduce (a9-a10), inputs (momenta,
weights) resident in HBM.  `e2e` is the same through heget_xsec_host with pinned HOST buffers
(H2D and D2H copies inside the timed region).  `pipeline` is the whole chain generated on the
device: heget_gen_events -> heget_amp2 -> heget_xsec_reduce inside one pair of CUDA events (the
analogue of the paper's timer, steps 2-6 of PAPER.md:116-122).  `per_config` repeats
the measurement for n = 2..8 in both precisions.  One JSON line is printed by rank 0.
"""
import argparse
import glob
import json
import math
import os
import re
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "events/s of summed |M|^2 for u ubar->n gamma"
UNIT = "events/s"
ALGOS = {"tree": 0, "subset": 1, "two-sided": 2}
THREAD_MAXN = 6     # n <= 5: one thread per event, n = 6: two / four lanes per event (csrc/amp2_thread.cu); n >= 7: one lane
                    # per helicity assignment (csrc/amp2.cu)


def kernel_name(algo, n):
    if algo == "tree":
        return "amp2_kernel" if n > THREAD_MAXN else ("amp2_thread%d_kernel" % n if n >= 5 else "amp2_thread_kernel")
    return {"subset": "amp2_subset_kernel", "two-sided": "amp2_twosided_kernel"}[algo]


# ---------------------------------------------------------------------------------------------
# flop models

def model_flops_per_event(n):
    """Model C of SURVEY 8(d): permutation tree with prefix reuse, Weyl form, the 2*2^n non-zero
    helicity assignments; 44 flop per internal node, 24 per leaf (FMA = 2)."""
    internal = sum(math.factorial(n) // math.factorial(n - l) for l in range(1, n))
    return 2 * 2 ** n * (44 * internal + 24 * math.factorial(n))


def executed_flops_per_event(n, precision="fp32"):
    """What the tree kernels execute per event, tables excluded.
    n >= 7 (lane per helicity assignment, factorised nodes psi = z v, csrc/amp2_chain.cuh): 2^n lanes;
    every ordered prefix of up to n-4 photons is rho (4 FMA) + the vector v of the node (5 FMA + 1 MUL)
    + the accumulation rho A (4 FMA) = 27 flop; a prefix of n-3 photons needs no vector (the rho of its
    three children come from the per-event rho table, their closing dots from the K table): rho +
    accumulation + three complex FMAs R K = 20 FMA = 40 flop.
    n <= 5 (thread per event, csrc/amp2_thread.cu): nodes are shared between helicity assignments (a
    prefix is evaluated once per helicity assignment of ITS photons): n = 5: per photon triple 12 vectors
    v2 and 6 v3 (11 flop), 48 rho (8), 24 products rho rho and 24 accumulations of Psi (16 each), 4 pair
    rows (32) and 32 closing dots (16 + 2), plus 10 v1 and 10 U (11); n = 4: 8 vectors v1 (11 flop),
    24 vectors v2 (11), 48 rho (8), 48 scalings/accumulations of psi_2 (16), 96 closing dots (16);
    n = 3: 6 vectors (11), 24 dots (16 + 2); n = 2: the closing rows only (counted with the tables).
    The kernels' whole count, tables included, is read from the SASS (sass_flops_per_event) or from the
    ncu summaries under profiles/."""
    if n >= 7:
        upper = sum(math.factorial(n) // math.factorial(n - l) for l in range(1, n - 3))
        return 2 ** n * (27 * upper + 40 * (math.factorial(n) // 6))
    if n == 6:
        # two lanes per event, 15 photon quadruples each: 12 (last, third) blocks of ~400 flop (10 vectors, 5 rho
        # tables, 8 products of two orderings, 8 accumulations), Psi 600, pair rows and 32 closing dots 912
        return 2 * 15 * (12 * 400 + 600 + 912)
    if n == 5:
        return 10 * (18 * 11 + 48 * 8 + 48 * 16 + 4 * 32 + 32 * 18) + 20 * 11
    if n == 4:
        return 8 * 11 + 24 * 11 + 48 * 8 + 48 * 16 + 96 * 16
    if n == 3:
        return 6 * 11 + 24 * 18
    return 0


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


_SASS_CACHE = {}
_SASS_DUMP = {}


def kernel_sass(kernel, n, precision):
    """The SASS lines of one amplitude kernel instantiation of the library that is loaded (cuobjdump), or None."""
    from paper_0908_4403_b200 import binding
    if "text" not in _SASS_DUMP:
        try:
            tool = "/usr/local/cuda/bin/cuobjdump" if os.path.exists("/usr/local/cuda/bin/cuobjdump") else "cuobjdump"
            _SASS_DUMP["text"] = subprocess.run([tool, "-sass", binding.LIB_PATH], capture_output=True, text=True,
                                                timeout=600).stdout.splitlines()
        except Exception:
            _SASS_DUMP["text"] = []
    t = "d" if precision == "fp64" else "f"
    want = "%sI%sE" % (kernel, t) if kernel in ("amp2_thread5_kernel", "amp2_thread6_kernel") else "%sILi%dE%s" % (kernel, n, t)
    body, on = [], False
    for line in _SASS_DUMP["text"]:
        if "Function :" in line:
            on = want in line
        elif on:
            body.append(line)
    return body or None


def kernel_sass_sha(kernel, n, precision):
    """sha256 over the instruction text of that kernel: what ties a committed ncu summary to a binary."""
    import hashlib
    body = kernel_sass(kernel, n, precision)
    if not body:
        return None
    text = "\n".join(l.strip() for l in body if re.match(r"\s+/\*[0-9a-f]{4,}\*/", l))
    return hashlib.sha256(text.encode()).hexdigest()[:16]


def sass_flops_per_event(n, precision):
    """Flops per event of the thread-per-event kernels (n <= 5), counted in the SASS of the library
    that is loaded: those kernels are straight-line code executed once per event (n = 5: plus one rolled
    loop over the 10 photon triples, whose body is weighted by its trip count), so the static count of
    {D,F}FMA (x2), {D,F}MUL, {D,F}ADD IS the executed count, tables included.  None if cuobjdump is not
    available or the control flow is not of that form."""
    if n > THREAD_MAXN:
        return None
    key = (n, precision)
    if key in _SASS_CACHE:
        return _SASS_CACHE[key]
    val = None
    try:
        body = kernel_sass(kernel_name("tree", n), n, precision) or []
        ops, loops, ok = [], [], True            # ops: (address, mnemonic); loops: (target, address of the backward branch)
        for l in body:
            m = re.match(r"\s+/\*([0-9a-f]{4,})\*/\s+(@!?U?P\d\s+)?([A-Z0-9_.]+)(.*?);", l)
            if not m:
                continue
            addr, pred, op, rest = int(m.group(1), 16), m.group(2), m.group(3), m.group(4)
            if op == "EXIT" and not pred:
                break                              # the slow paths of division and square root and the padding follow
            if op.startswith("BRA"):
                t = re.search(r"0x([0-9a-f]+)", rest)
                ok = ok and bool(t)
                if t and int(t.group(1), 16) <= addr:
                    loops.append((int(t.group(1), 16), addr))     # forward branches only skip a slow-path call
            ops.append((addr, op.split(".")[0]))
        # n <= 4: no loop at all; n = 5, 6: the rolled loop over the 10 photon triples / 15 quadruples; the fp64
        # 6-photon kernel also keeps its loop over the 62 subsets rolled, two per trip.  Loops in program order.
        trips = {(5, "fp64"): [10], (5, "fp32"): [10], (6, "fp32"): [15], (6, "fp64"): [31, 15]}.get((n, precision), [])
        lanes = {6: 4 if precision == "fp64" else 2}.get(n, 1)      # lanes per event (HEGET_THREAD6_FIX64 / FIX32)
        loops.sort(key=lambda lp: lp[1])
        nested = any(a[0] <= b[0] <= a[1] for a in loops for b in loops if a is not b)
        if ops and ok and len(loops) == len(trips) and not nested:
            w = {"DFMA": 2, "FFMA": 2, "DMUL": 1, "FMUL": 1, "DADD": 1, "FADD": 1}
            mult = lambda a: next((tr for (lo, hi), tr in zip(loops, trips) if lo <= a <= hi), 1)
            val = float(lanes * sum(w.get(o, 0) * mult(a) for a, o in ops))
    except Exception:
        val = None
    _SASS_CACHE[key] = val
    return val


def ncu_summary(config, precision, kernel, measured_ms, events, n):
    """The committed `ncu --set full` summary of this kernel under profiles/ (newest round first):
    counted flops per event, DRAM bytes per launch and the kernel time of the capture.  The summary
    describes the binary it was captured from: it is used only if it names the kernel that runs now, was
    taken on the same number of events, carries the SASS hash of THIS library's kernel (`sass_sha256:`
    line; kernel_sass_sha) and its duration agrees with the one measured here within 5 % (or 4 us: CUDA
    events around a kernel of a few microseconds include its launch latency, ncu's duration does not);
    otherwise the status says why and the caller falls back to what it can measure itself."""
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_amp2_%s_%s.txt" % (config, precision))), reverse=True)
    if not files:
        return {"status": "no summary under profiles/ for %s %s" % (config, precision)}
    text = open(files[0]).read()
    name = os.path.relpath(files[0], ROOT)
    m_kernel = re.search(r"^kernel: .*?(\w+)<", text, re.M)
    m_time = re.search(r"gpu__time_duration\.sum\s+([0-9.,]+)\s*(us|ms|ns|s)\b", text)
    m_flop = re.search(r"=\s*([0-9.eE+]+) flop per event", text)
    m_ev = re.search(r"/\s*(\d+) events", text)
    scale = {"ns": 1e-6, "us": 1e-3, "ms": 1.0, "s": 1e3}
    unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    dram = 0.0
    for key in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
        m = re.search(re.escape(key) + r"\s+([0-9.,]+)\s*(\w+)", text)
        if not m or m.group(2) not in unit:
            return {"status": "STALE: %s has no %s" % (name, key), "file": name}
        dram += float(m.group(1).replace(",", "")) * unit[m.group(2)]
    if not (m_kernel and m_time and m_flop and m_ev):
        return {"status": "STALE: %s is not a summary this parser understands" % name, "file": name}
    ms = float(m_time.group(1).replace(",", "")) * scale[m_time.group(2)]
    out = {"file": name, "kernel": m_kernel.group(1), "kernel_ms": ms, "flops_per_event": float(m_flop.group(1)),
           "dram_bytes": dram, "events": int(m_ev.group(1))}
    if out["kernel"] != kernel:
        out["status"] = "STALE: %s is a capture of %s, the kernel that runs is %s" % (name, out["kernel"], kernel)
    elif out["events"] != events:
        out["status"] = "STALE: %s was captured on %d events, this run has %d" % (name, out["events"], events)
    else:
        m_sha = re.search(r"^sass_sha256: ([0-9a-f]+)", text, re.M)
        sha = kernel_sass_sha(kernel, n, precision)
        out["sass_sha256"] = sha
        if not m_sha or sha is None or m_sha.group(1) != sha:
            out["status"] = "STALE: %s was captured from a different binary of %s (SASS hash %s, loaded library %s)" % (
                name, kernel, m_sha.group(1) if m_sha else "missing", sha)
        elif abs(ms / measured_ms - 1.0) > 0.05 and abs(ms - measured_ms) > 0.004:
            # the same instructions ran (hash), so the counted flops and bytes per event hold; the clock or the
            # neighbours of this launch differ from the capture's
            out["status"] = "ok (same SASS as the capture; duration there %.4f ms, here %.4f ms)" % (ms, measured_ms)
            out["duration_agrees"] = False
        else:
            out["status"] = "ok"
            out["duration_agrees"] = True
    if not out["status"].startswith("ok"):
        sys.stderr.write("bench.py: " + out["status"] + "\n")
    return out


def theoretical_peak(precision, sm_count, sm_max_mhz):
    lanes = 128 if precision == "fp32" else 64       # FP32 / FP64 FMA lanes per SM on B200
    return sm_count * lanes * 2 * sm_max_mhz * 1e6


# ---------------------------------------------------------------------------------------------
# clocks

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


# ---------------------------------------------------------------------------------------------
# CPU baseline: the oracle as it stands, on the host cores

# rough oracle<double> cost per event in core-seconds (sizes the one-second pilot only)
ORACLE_CORE_S = {2: 2e-6, 3: 2.5e-5, 4: 5e-4, 5: 1e-2, 6: 0.4, 7: 7.0, 8: 130.0}


def oracle_sample_events(cfg, seconds_budget=12.0):
    """How many events of this config the oracle is timed on: a BOUNDED sample sized for about
    `seconds_budget` seconds of wall time on this host, from a pilot run of the oracle itself."""
    cores = os.cpu_count() or 1
    pilot = max(min(int(1.0 * cores / ORACLE_CORE_S[cfg["n"]]), cfg["N"]), 1)
    if ORACLE_CORE_S[cfg["n"]] / cores > seconds_budget / 2:
        return 1      # one event is already most of the budget (the oracle spreads its helicity assignments over the cores)
    rate, _, _ = time_oracle(cfg, pilot)
    return max(min(int(rate * seconds_budget), cfg["N"]), 1)


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


def cpu_baseline(name, cfg, seconds_budget):
    n_ev = oracle_sample_events(cfg, seconds_budget)
    v, dt, cores = time_oracle(cfg, n_ev)
    return {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "first %d of %d events of %s, oracle<double>, %.1f s" % (n_ev, cfg["N"], name, dt)}


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


# ---------------------------------------------------------------------------------------------

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
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=hg.device)   # > 126 MB L2
    PREC = {"fp64": FP64, "fp32": FP32}

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def gen(c, nl, first, momenta=None, weight=None):
        return hg.gen_events(c["seed"], c["n"], nl, mode=c["mode"], a=c["a"], b=c["b"], y_max=c["y_max"],
                             apply_cuts=c["apply_cuts"], first_event=first, momenta=momenta, weight=weight)

    def timed_run(name, precision, steps, warmup, algo=0, pipeline=False):
        """Device-timed steps on resident inputs: heget_amp2 + heget_xsec_reduce (+ the all-reduce of
        the three sums for world > 1), or with pipeline=True heget_gen_events + both, CUDA events on the
        launching stream.  Weak scaling: every rank processes the config's full per-GPU batch on its own
        contiguous range of global event indices.  Returns total ms over the steps, the mean and
        best amp2-kernel ms, the three sums and the events per rank."""
        c = workloads.CONFIGS[name]
        nl, first = c["N"], rank * c["N"]
        mom, w = gen(c, nl, first)
        amp2 = torch.empty(nl, dtype=torch.float64, device=hg.device)
        out3 = torch.empty(3, dtype=torch.float64, device=hg.device)

        def step(ev=None):
            if ev:
                ev[0].record()
            if pipeline:
                gen(c, nl, first, mom, w)
            if ev:
                ev[1].record()
            hg.amp2(mom, PREC[precision], out=amp2, algo=algo)
            if ev:
                ev[2].record()
            hg.xsec_reduce(amp2, w, c["n"], out3=out3)
            if world > 1:
                dist.all_reduce(out3)              # the only exchange of the path, inside the timed window
            if ev:
                ev[3].record()

        for _ in range(warmup):
            step()
        barrier()
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(steps)]
        for ev in evs:
            flush_buf.zero_()                      # L2 flush, outside the timed events
            step(ev)
        barrier()
        step_ms = [e[0].elapsed_time(e[3]) for e in evs]
        amp_ms = [e[1].elapsed_time(e[2]) for e in evs]
        gen_ms = [e[0].elapsed_time(e[1]) for e in evs]
        return {"total_ms": sum(step_ms), "step_ms": sum(step_ms) / steps, "amp_ms": sum(amp_ms) / steps,
                "amp_ms_best": min(amp_ms), "gen_ms": sum(gen_ms) / steps, "sums": out3.cpu().numpy(), "events": nl}

    def max_over_ranks(x):
        if world > 1:
            t = torch.tensor([x], dtype=torch.float64, device=hg.device)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            return t.item()
        return x

    # ---- headline: amp2 + reduce on resident inputs
    launches0 = hg.launch_count()
    sampler = ClockSampler(local_rank)
    sampler.start()
    head = timed_run(args.config, args.precision, args.steps, args.warmup, algo=ALGOS[args.algo])
    clocks = sampler.stop()
    launches = hg.launch_count() - launches0 - 3 * args.warmup - 1   # minus warm-up steps and the generator
    nl = head["events"]
    total_ms = max_over_ranks(head["total_ms"])
    value = world * nl * args.steps / (total_ms * 1e-3)
    amp_ms, amp_ms_best, sums = head["amp_ms"], head["amp_ms_best"], head["sums"]

    # ---- pipeline: gen + amp2 + reduce in one event pair (device-generated inputs, nothing crosses PCIe)
    pipe = timed_run(args.config, args.precision, max(1, min(args.steps, 5)), 3, algo=ALGOS[args.algo], pipeline=True)
    pipe_ms = max_over_ranks(pipe["step_ms"])

    # ---- end to end through the host-buffer entry point (pinned host inputs, H2D + D2H inside)
    mom_d, w_d = gen(cfg, nl, rank * nl)
    mom_h = torch.empty(mom_d.shape, dtype=torch.float64).pin_memory()
    w_h = torch.empty(w_d.shape, dtype=torch.float64).pin_memory()
    mom_h.copy_(mom_d)
    w_h.copy_(w_d)
    out3_h = torch.empty(3, dtype=torch.float64).pin_memory()
    prec = PREC[args.precision]
    for _ in range(3):       # warm-up, and the staging buffers of heget_xsec_host are allocated here
        hg.xsec_host(mom_h, w_h, prec, out3=out3_h)
    barrier()
    e2e_steps = max(1, min(args.steps, 5))
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        hg.xsec_host(mom_h, w_h, prec, out3=out3_h)
        if world > 1:
            t3 = out3_h.to(hg.device)
            dist.all_reduce(t3)
            out3_h.copy_(t3)
    barrier()
    e2e_s = max_over_ranks(time.perf_counter() - t0)
    e2e_value = world * nl * e2e_steps / e2e_s

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (amp2): plain-ALU bound.  `achieved` = flops the kernel
    # executes (the ncu-counted figure is the %peak figure) over its own time, measured
    # here with CUDA events; model C (the survey's algorithmic count, which ignores the parity relation,
    # the normalised E' entries and the sharing of prefixes between helicity assignments) over the
    # same time is given beside it as the cross-check.
    props = torch.cuda.get_device_properties(local_rank)
    sm_max = clocks["sm_max_mhz"] or 1965.0
    peaks = {p: {"measured": hg.fma_peak(PREC[p], 0), "three_reg": hg.fma_peak(PREC[p], 1), "node": hg.fma_peak(PREC[p], 2),
                 "theory": theoretical_peak(p, props.multi_processor_count, sm_max)} for p in ("fp64", "fp32")}

    def flops_of(name, nph, precision, algo, ms, events):
        """(flops per event, source, ncu summary or None) for one kernel of this run."""
        summ = ncu_summary(name, precision, kernel_name(algo, nph), ms, events, nph) if algo == "tree" else None
        if summ and summ["status"].startswith("ok"):
            return summ["flops_per_event"], "ncu-counted over the whole kernel, tables included (%s)" % summ["file"], summ
        sass = sass_flops_per_event(nph, precision) if algo == "tree" else None
        if sass:
            return sass, "counted in the SASS of the loaded library (straight-line kernel, one pass per event, tables included)", summ
        return (executed_flops_per_event_algo(nph, algo, precision),
                "executed-instruction model of the tree, tables (< 1 % from 6 photons on) excluded", summ)

    pk = peaks[args.precision]
    fpe, fsrc, summ = flops_of(args.config, n, args.precision, args.algo, amp_ms, nl)
    tree_model = executed_flops_per_event_algo(n, args.algo, args.precision)
    achieved = fpe * nl / (amp_ms * 1e-3)
    model_c = model_flops_per_event(n) * nl / (amp_ms * 1e-3)
    bytes_alg = nl * ((n + 2) * 32 + 8)
    roofline = {"bound": "alu", "achieved": achieved / 1e12, "peak": pk["measured"] / 1e12, "unit": "TFLOP/s",
                "frac": achieved / pk["measured"],
                "traffic": summ["dram_bytes"] if summ and summ["status"].startswith("ok") else None,
                "kernel": "%s<%d,%s>" % (kernel_name(args.algo, n), n, "double" if prec == FP64 else "float"),
                "kernel_ms": amp_ms, "kernel_ms_best": amp_ms_best,
                "flops_per_event": fpe, "flops_source": fsrc,
                "ncu_summary": ({k: summ[k] for k in ("status", "file", "kernel_ms", "sass_sha256", "duration_agrees") if k in summ} if summ else None),
                "flops_per_event_tree_model": tree_model,
                "tree_model_tflops": tree_model * nl / (amp_ms * 1e-3) / 1e12,
                "peak_source": "heget_fma_peak on this GPU: FMA with constant-bank operands "
                               "(MEASURED_PEAKS.json has no non-tensor figure)",
                "peak_theoretical": pk["theory"] / 1e12, "frac_of_theoretical": achieved / pk["theory"],
                "peak_three_register_fma": pk["three_reg"] / 1e12, "peak_node_pattern": pk["node"] / 1e12,
                "frac_of_node_pattern": achieved / pk["node"],
                "model_c_tflops": model_c / 1e12, "model_c_frac": model_c / pk["measured"],
                "algorithmic_bytes": bytes_alg, "hbm_gbs": bytes_alg / (amp_ms * 1e-3) / 1e9,
                "frac_note": "frac counts EXECUTED flops (what ncu counts); model_c_frac counts SURVEY 8(d)'s fixed "
                             "algorithmic figure (model C) over the same time.  Work removed by the parity relation, by "
                             "sharing prefixes between helicity assignments and by re-associating factors lowers frac "
                             "while events/s and model_c_frac rise"}

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
              "pipeline": {"value": world * nl / (pipe_ms * 1e-3), "unit": UNIT, "ms_per_step": pipe_ms,
                           "gen_ms": pipe["gen_ms"], "amp2_ms": pipe["amp_ms"],
                           "what": "heget_gen_events + heget_amp2 + heget_xsec_reduce inside one CUDA-event pair"},
              "gpu_launches": int(launches),
              "roofline": roofline,
              "xsec": {"sum_wA": float(sums[0]), "sum_wA2": float(sums[1]), "n_pass": float(sums[2])}}

    if not args.no_cpu_baseline:
        result["cpu_baseline"] = cpu_baseline(args.config, cfg, 12.0)

    if not args.no_sweep and world == 1:
        table = []
        for name in workloads.ORDER:
            c = workloads.CONFIGS[name]
            nph = c["n"]
            cpu = None if args.no_cpu_baseline else cpu_baseline(name, c, 3.0)
            for precision in ("fp32", "fp64"):
                pkk = peaks[precision]
                for algo_name, note in (
                        ("tree", None),
                        ("subset", "HEGET_ALGO_SUBSET (heget_amp2_algo): not the permutation tree, own flop count"),
                        ("two-sided", "HEGET_ALGO_TREE2 (heget_amp2_algo): tree from u to depth n-4, closed with "
                                      "row vectors chained from ubar; own flop count")):
                    r = timed_run(name, precision, 3, 3, algo=ALGOS[algo_name])
                    ms, nn = r["amp_ms"], r["events"]
                    row = {"workload": name, "n": nph, "precision": precision, "events": nn, "algo": algo_name,
                           "amp2_ms": ms, "amp2_ms_best": r["amp_ms_best"], "events_per_s": nn / (ms * 1e-3)}
                    model = executed_flops_per_event_algo(nph, algo_name, precision)
                    row["executed_tflops"] = model * nn / (ms * 1e-3) / 1e12
                    if algo_name == "tree":
                        f, src, s = flops_of(name, nph, precision, "tree", ms, nn)
                        p = timed_run(name, precision, 3, 3, pipeline=True)
                        row.update({"counted_tflops": f * nn / (ms * 1e-3) / 1e12, "flops_per_event": f, "flops_source": src,
                                    "frac_of_measured_peak": f * nn / (ms * 1e-3) / pkk["measured"],
                                    "frac_of_theoretical_peak": f * nn / (ms * 1e-3) / pkk["theory"],
                                    "model_c_tflops": model_flops_per_event(nph) * nn / (ms * 1e-3) / 1e12,
                                    "hbm_gbs": nn * ((nph + 2) * 32 + 8) / (ms * 1e-3) / 1e9,
                                    "pipeline_ms": p["step_ms"], "gen_ms": p["gen_ms"],
                                    "pipeline_events_per_s": nn / (p["step_ms"] * 1e-3)})
                        if cpu:
                            row["cpu_baseline"] = cpu
                    else:
                        row.update({"frac_of_measured_peak": model * nn / (ms * 1e-3) / pkk["measured"], "note": note})
                    table.append(row)
        result["per_config"] = table

        # 2 photons are HBM- and launch-latency bound (136 B and ~340 flop per event): the same kernel on 2^20
        # events against the measured HBM copy rate, beside config 1's 65,536 events (a few microseconds,
        # i.e. the launch-latency floor)
        hbm = _hbm_peak()
        c2 = workloads.CONFIGS["2gamma"]
        rows2 = []
        for n2 in (c2["N"], 1 << 20, 1 << 23):
            m2, _ = hg.gen_events(c2["seed"], 2, n2, mode=c2["mode"], a=c2["a"])
            o2 = torch.empty(n2, dtype=torch.float64, device=hg.device)
            for _ in range(3):
                hg.amp2(m2, FP64, out=o2)
            ts = []
            for _ in range(7):
                flush_buf.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                hg.amp2(m2, FP64, out=o2)
                e1.record()
                torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            ms2 = sorted(ts)[len(ts) // 2]
            rows2.append({"events": n2, "amp2_ms": ms2, "events_per_s": n2 / (ms2 * 1e-3),
                          "hbm_gbs": n2 * 136 / (ms2 * 1e-3) / 1e9, "frac_of_hbm_peak": n2 * 136 / (ms2 * 1e-3) / 1e9 / hbm["value"]})
        result["two_photon_hbm"] = {"bytes_per_event": 136, "hbm_peak_gbs": hbm, "precision": "fp64", "rows": rows2}
        result["peaks_tflops"] = {p: {k: v / 1e12 for k, v in d.items()} for p, d in peaks.items()}
        result["hbm_peak_gbs"] = _hbm_peak()

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
        result["next1"] = {"amp2_sampled_ms": ev[0].elapsed_time(ev[1]),
                           "amp2_sampled_events_per_s": nl / (ev[0].elapsed_time(ev[1]) * 1e-3),
                           "histogram_ms": ev[1].elapsed_time(ev[2]), "events": nl, "precision": args.precision}

    print(json.dumps(result))
    hg.close()


def _hbm_peak():
    """Measured HBM copy rate of this pool's B200s (driver-written MEASURED_PEAKS.json), else the
    fallback of the profiling guide."""
    try:
        return {"value": json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"], "source": "MEASURED_PEAKS.json"}
    except Exception:
        return {"value": 6540.0, "source": "fallback: B200_PROFILING.md"}


if __name__ == "__main__":
    main()
