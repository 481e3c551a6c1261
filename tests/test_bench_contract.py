"""bench.py's reference arm (the CPU oracle on the host cores) runs without a GPU: its JSON line
must carry the keys the driver's contract names, and the flop models bench.py reports must agree
with the node counts of SURVEY 8(a)."""
import json
import math
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", "--config", "2gamma"], capture_output=True, text=True, timeout=600,
                         env=dict(os.environ, RANK="0", WORLD_SIZE="1"))
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                "scaling", "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in line, key
    assert line["impl"] == "reference" and line["unit"] == "events/s" and line["value"] > 0
    assert line["config"]["workload"] == "2gamma" and line["vs_baseline"] is None
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0


def test_other_ranks_of_the_reference_arm_exit_silently():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", "--config", "2gamma", "--gpus", "2"], capture_output=True, text=True,
                         timeout=600, env=dict(os.environ, RANK="1", WORLD_SIZE="2"))
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_flop_models_match_the_node_counts_of_the_survey():
    sys.path.insert(0, ROOT)
    import bench
    internal = {2: 2, 3: 9, 4: 40, 5: 205, 6: 1236, 7: 8659, 8: 69280}
    for n, nodes in internal.items():
        assert bench.model_flops_per_event(n) == 2 * 2 ** n * (44 * nodes + 24 * math.factorial(n))
        upper = nodes - math.factorial(n)            # prefixes of up to n-2 photons
        if n >= 7:   # lane per helicity assignment: 27 flop per factorised node down to n-4 photons, 40 per node of n-3
            deep2, deep3 = math.factorial(n) // 2, math.factorial(n) // 6     # prefixes of exactly n-2 / n-3 photons
            assert bench.executed_flops_per_event(n, "fp32") == 2 ** n * (27 * (upper - deep2 - deep3) + 40 * deep3)
        else:        # thread per event: prefixes shared between helicity assignments, far below one tree per assignment
            assert bench.executed_flops_per_event(n, "fp32") < 2 ** n * (27 * upper + 8 * math.factorial(n)) or n == 2
        for algo in ("subset", "two-sided"):
            # never more work than the one-sided tree once there is a tree to speak of (at n = 4 the
            # tree kernel shares its first two levels between lanes and its tables are not counted)
            assert 0 < bench.executed_flops_per_event_algo(n, algo)
            if n >= 6:
                assert bench.executed_flops_per_event_algo(n, algo) <= bench.executed_flops_per_event(n, "fp32")
    # model C as tabulated in SURVEY 8(d): 1.09e3, 7.5e4, 2.06e9 flop per event
    assert abs(bench.model_flops_per_event(2) / 1.09e3 - 1) < 0.01
    assert abs(bench.model_flops_per_event(4) / 7.5e4 - 1) < 0.01
    assert abs(bench.model_flops_per_event(8) / 2.06e9 - 1) < 0.01


import pytest


@pytest.mark.gpu
def test_headline_line_carries_the_contract_and_a_fresh_ncu_summary():
    """python bench.py (headline config, no sweep): the JSON line has every key the driver's contract names,
    the roofline numerator comes from a committed ncu summary of THE kernel that ran (status ok: same kernel,
    same event count, duration within 5 % of the one measured in this run), and its DRAM traffic is the
    algorithmic traffic, not more."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "5", "--warmup", "3", "--no-sweep",
                          "--no-cpu-baseline"], capture_output=True, text=True, timeout=900)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "pipeline", "gpu_launches", "roofline"):
        assert key in line, key
    assert line["config"]["workload"] == "4gamma" and line["dtype"] == "f64" and line["vs_baseline"] is None
    assert line["gpu_launches"] == 3 * 5 and line["value"] > 1e9
    assert line["e2e"]["h2d_bytes_per_step"] == (1 << 20) * (6 * 32 + 8) and 0 < line["e2e"]["value"] < line["value"]
    assert 0 < line["pipeline"]["value"] < line["value"]
    r = line["roofline"]
    assert r["bound"] == "alu" and r["kernel"].startswith("amp2_thread_kernel<4,double>")
    assert r["ncu_summary"]["status"] == "ok" and r["ncu_summary"]["duration_agrees"], r["ncu_summary"]
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and 0.3 < r["frac"] < 1.0
    assert 0.9 < r["traffic"] / r["algorithmic_bytes"] < 1.1
    # the SASS count of the loaded library and the ncu-counted figure describe the same straight-line kernel
    sys.path.insert(0, ROOT)
    import bench
    assert abs(bench.sass_flops_per_event(4, "fp64") / r["flops_per_event"] - 1.0) < 0.01


def test_committed_ncu_summaries_describe_the_kernels_built_from_this_source():
    """Every profiles/r02_amp2_<config>_<precision>.txt carries the hash of the SASS of the kernel it was captured
    from; the library built from the source at hand must contain exactly that kernel (the build is deterministic),
    otherwise the summary is stale and bench.py would refuse it."""
    import re
    sys.path.insert(0, ROOT)
    import bench
    from paper_0908_4403_b200 import build, workloads
    build.build()
    if bench.kernel_sass("amp2_kernel", 8, "fp64") is None:
        pytest.skip("cuobjdump is not available: the SASS of the library cannot be read")
    for name in workloads.ORDER:
        n = workloads.CONFIGS[name]["n"]
        for precision in ("fp64", "fp32"):
            text = open(os.path.join(ROOT, "profiles", "r02_amp2_%s_%s.txt" % (name, precision))).read()
            m = re.search(r"^sass_sha256: ([0-9a-f]+)", text, re.M)
            assert m, (name, precision)
            kernel = bench.kernel_name("tree", n)
            assert re.search(r"^kernel: .*?%s<" % kernel, text, re.M), (name, precision, kernel)
            assert bench.kernel_sass_sha(kernel, n, precision) == m.group(1), (name, precision)
