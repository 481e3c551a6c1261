"""Writes tests/golden/amp2_<config>.npz: the ORACLE's summed |M|^2 on the event subsets that
BASELINE.json `configs` name ("the CPU oracle runs on a 4,096-event subset" at 7 gamma, "on a
512-event subset" at 8 gamma; 2,048 events at 6 gamma), PAPER.md:256 ("compared ... for all
helicities at many points" is the paper's own validation standard).

Calls only `oracle/` (plus the plain workload parameters of workloads.py, loaded by path so that
nothing of the CUDA package is imported).  Nothing here comes from the CUDA path.

Per config the file holds
  momenta[N][n+2][4], weight[N]   the first N events of the config from the oracle's generator
  amp2_d[N]                       oracle<double> on every event
  amp2_ld[N]                      oracle<long double> (rounded to double) on the events marked
  has_ld[N]                       in has_ld: all cut-passing events (weight != 0), where the
                                  1e-12 gate binds (reading R14); NaN elsewhere
  momenta_sha256                  of momenta.tobytes(), so a test can tell a regenerated set

The work is tens of core-hours at 8 gamma, so it is cut into parts that are written to
--parts-dir as they finish; rerunning skips finished parts and `--merge` assembles the .npz.

  python tests/golden/make_amp2_golden.py --config 7gamma            # all parts, then merge
  python tests/golden/make_amp2_golden.py --config 8gamma --kind ld --part-range 0 4
  python tests/golden/make_amp2_golden.py --config 8gamma --merge
"""
import argparse
import hashlib
import importlib.util
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402

_spec = importlib.util.spec_from_file_location(
    "heget_workloads", os.path.join(ROOT, "paper_0908_4403_b200", "workloads.py"))
workloads = importlib.util.module_from_spec(_spec)
_spec.loader.exec_module(workloads)

# config -> (events, events per part)
SUBSETS = {"6gamma": (2048, 256), "7gamma": (4096, 128), "8gamma": (512, 16)}


def events(name):
    c = workloads.CONFIGS[name]
    N = SUBSETS[name][0]
    return oracle.gen_events(c["seed"], c["n"], N, mode=c["mode"], a=c["a"], b=c["b"], y_max=c["y_max"],
                             apply_cuts=c["apply_cuts"], pt_cut=workloads.PT_CUT, eta_cut=workloads.ETA_CUT,
                             dr_cut=workloads.DR_CUT, first_event=0)


def part_path(parts_dir, name, kind, k):
    return os.path.join(parts_dir, "%s_%s_%04d.npy" % (name, kind, k))


def run_parts(name, kind, parts_dir, lo, hi):
    mom, w = events(name)
    N, per = SUBSETS[name]
    nparts = N // per
    os.makedirs(parts_dir, exist_ok=True)
    for k in range(max(lo, 0), min(hi, nparts)):
        path = part_path(parts_dir, name, kind, k)
        if os.path.exists(path):
            continue
        sl = slice(k * per, (k + 1) * per)
        out = np.full(per, np.nan)
        sel = np.ones(per, bool) if kind == "d" else (w[sl] != 0)
        t0 = time.time()
        if sel.any():
            out[sel] = oracle.amp2(mom[sl][sel], extended=(kind == "ld"))
        np.save(path + ".tmp.npy", out)
        os.replace(path + ".tmp.npy", path)
        print("%s %s part %d/%d: %d events, %.1f s, %d threads" % (name, kind, k, nparts, int(sel.sum()),
                                                                     time.time() - t0, oracle.num_threads()),
              flush=True)


def merge(name, parts_dir):
    mom, w = events(name)
    N, per = SUBSETS[name]
    got = {}
    for kind in ("d", "ld"):
        parts = []
        for k in range(N // per):
            path = part_path(parts_dir, name, kind, k)
            if not os.path.exists(path):
                raise SystemExit("missing part %s" % path)
            parts.append(np.load(path))
        got[kind] = np.concatenate(parts)
    has_ld = w != 0
    assert np.all(np.isfinite(got["d"])) and np.all(np.isfinite(got["ld"][has_ld]))
    assert np.all(np.isnan(got["ld"][~has_ld]))
    out = os.path.join(HERE, "amp2_%s.npz" % name)
    np.savez(out, momenta=mom, weight=w, amp2_d=got["d"], amp2_ld=got["ld"], has_ld=has_ld,
             momenta_sha256=np.array(hashlib.sha256(mom.tobytes()).hexdigest()))
    ladder = np.abs(got["d"][has_ld] / got["ld"][has_ld] - 1.0)
    print("%s: %d events, %d cut-passing; oracle<double> vs oracle<long double> on those: max %.3e median %.3e"
          % (name, N, int(has_ld.sum()), ladder.max(), np.median(ladder)))
    print("wrote", out)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", required=True, choices=sorted(SUBSETS))
    ap.add_argument("--kind", choices=["d", "ld", "both"], default="both")
    ap.add_argument("--part-range", type=int, nargs=2, default=[0, 1 << 30])
    ap.add_argument("--parts-dir", default="/tmp/heget_golden_parts")
    ap.add_argument("--merge", action="store_true", help="only assemble the .npz from finished parts")
    a = ap.parse_args()
    if not a.merge:
        for kind in (("d", "ld") if a.kind == "both" else (a.kind,)):
            run_parts(a.config, kind, a.parts_dir, *a.part_range)
    if a.merge or (a.kind == "both" and a.part_range == [0, 1 << 30]):
        merge(a.config, a.parts_dir)


if __name__ == "__main__":
    main()
