"""Host-side checks of the constant index tables compiled into the thread-per-event kernels
(csrc/amp2_thread.cu): the kernels index their shared-memory columns by the position of an entry in these
tables (colex rank of a photon triple, rank of a photon pair), so a wrong row would read another subset's
propagator entry.  compute-sanitizer is not available on the GPU pool; this is the part of that
addressing that can be checked without a GPU."""
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = open(os.path.join(ROOT, "paper_0908_4403_b200", "csrc", "amp2_thread.cu")).read()


def table(name):
    m = re.search(name + r"\[\d+\]\s*=\s*\{(.*?)\};", SRC, re.S)
    assert m, name
    return [int(x) for x in re.findall(r"\d+", m.group(1))]


def test_triples_of_the_five_photon_kernel():
    flat = table("c_triples5")
    rows = [flat[5 * r: 5 * r + 5] for r in range(10)]
    assert len(flat) == 50
    for rank, (i, j, k, a, b) in enumerate(rows):
        assert i < j < k and a < b and sorted((i, j, k, a, b)) == [0, 1, 2, 3, 4]
        assert k * (k - 1) * (k - 2) // 6 + j * (j - 1) // 2 + i == rank      # P3 slot = colex rank of the triple


def test_quadruples_of_the_six_photon_kernel():
    flat = table("c_quads6")
    rows = [flat[6 * r: 6 * r + 6] for r in range(15)]
    assert len(flat) == 90
    for rank, (t0, t1, t2, t3, a, b) in enumerate(rows):
        assert t0 < t1 < t2 < t3 and a < b and sorted((t0, t1, t2, t3, a, b)) == [0, 1, 2, 3, 4, 5]
        assert b * (b - 1) // 2 + a == rank                                    # P4 slot = rank of the complementary pair


def test_column_layout_of_the_six_photon_kernel_has_no_overlap():
    m = re.search(r"struct Col6 \{.*?E = (\d+), P1 = (\d+), P5 = (\d+), P2 = (\d+), P3 = (\d+), P4 = (\d+), AMP = 2 \* (\d+);", SRC, re.S)
    assert m
    e, p1, p5, p2, p3, p4, slots = map(int, m.groups())
    sizes = [(e, 6), (p1, 6), (p5, 6), (p2, 15), (p3, 20), (p4, 15)]          # photons, C(6,2), C(6,3), C(6,4)
    end = 0
    for start, count in sizes:
        assert start == end
        end = start + count
    assert end == slots
