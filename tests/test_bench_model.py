"""bench.py's roofline denominators: the stored flop model equals the oracle's counted operations, the byte
model equals the array sizes; the JSON helpers work without a GPU."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402
from paper_2210_17509_b200 import inputs  # noqa: E402


@pytest.mark.parametrize("recon", ["weno5", "minmod", "mc"])
def test_flop_model_matches_oracle_count(oracle, recon):
    for n in ((20, 20, 20), (24, 12, 8)):
        prob = inputs.general_metric_box(n=n, seed=2) if n[0] != n[1] else inputs.sweep_boxes(n[0], 1)
        _, ops = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma,
                                     variant="count")
        counted = sum(ops.values()) / prob.cells
        model = bench.algorithmic_flops_per_cell(n, recon)
        assert model == pytest.approx(counted, rel=0.01), (n, recon, counted, model)


def test_byte_model():
    assert bench.algorithmic_bytes_per_cell((256, 256, 256), 3) == pytest.approx(269.8, abs=0.1)
    assert bench.algorithmic_bytes_per_cell((32, 32, 32), 3) == pytest.approx(385.5, abs=0.1)
    assert bench.FP64_PEAK_NOMINAL_TFLOPS == pytest.approx(37.2, abs=0.05)


def test_sub_block_is_a_view_of_the_workload():
    prob = inputs.sweep_boxes(16, 2)
    (p, m, k), n = bench._sub_block(prob, 5, 7, 9)
    assert n == (9, 7, 5) and p.shape == (1, 8, 11, 13, 15) and m.shape[1] == 10 and k.shape[1] == 6
    assert np.array_equal(p[0, :, :, :, :], prob.prim[0, :, :11, :13, :15])


def test_rank_workloads_differ_but_share_shape():
    a = bench.load_workload("c5-32", 0)
    b = bench.load_workload("c5-32", 1)
    assert a.prim.shape == b.prim.shape and not np.array_equal(a.prim[0], b.prim[0])
    assert np.array_equal(a.prim[0], inputs.sweep_boxes(32, 1).prim[0])
