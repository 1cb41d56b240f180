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


# Hand counts of the oracle's pieces, derived by reading the formulas of SURVEY.md section 8.c.1 / oracle/valencia_oracle.cpp
# line by line (add = sub = mul = div = sqrt = 1; compares, selects, sign flips, abs, min/max are free):
#   recon_weno5 (O2): three smoothness indicators 12 + 9 + 12 = 33; three candidates per face
#       (3 mul 2 add 1 div) + 2 x (2 mul 2 add 1 div) = 16; combination: 3 (eps + beta) + 3 x (mul, div) + 5 (numerator)
#       + 2 (denominator) + 1 (quotient) = 17;   33 + 2 x (16 + 17) = 99
#   recon_minmod: 2 differences, their product, 2 x (0.5 sigma, +-) = 7;   MC adds 2|dm|, 2|dp|, |dm+dp|/2 = 4 when the
#       slopes agree in sign (data dependent)
#   face average (O1): 10 x (add, mul) = 20
#   metric_complete_face: 3 cofactors x 3 + determinant 5 + sqrt + the dd cofactor (0 for x, 3 for y and z) + 1 div = 16 / 19
#   admissible (O3): v_i 3 x 5, v^2 5 = 20
#   prim2con_point (O4): v_i 15, v^2 5, W 3, B_i 15, B^2 5, B.v 5, alpha b^0 1, b^2 4, b_i 9, p 3, rho h 3, rho h* 1, P* 2, W^2 1,
#       D 2, S_j 3 x 5, tau 6, calB 3 = 98
#   flux_point (O5): vtilde 6, sqrt(gamma) P* 1, calB^d/W 1, F_D 2, F_S 3 x 4 + 1, F_tau 6, F_B 3 x 4 = 41
#   wavespeeds_point (O6): c_s^2 2, v_A^2 1, a^2 3, 1 - v^2 a^2 2, discriminant 8, sqrt 1, 2 x 6 = 29
#   hlle (O7): 8 x 9 = 72
#   flux difference (O7): (F - F)/dx, acc -= : 3 per component
#   derivative (O8): 8 (m - m), (m - m), -, 12 dx, / = 6
#   metric_complete: 6 cofactors x 3, determinant 5, sqrt, 6 div = 30
#   sources_point (O9): metric_complete 30, prim2con 98, W^2 1, vtilde 6, b^i 9, T00 6, T0i 3 x 10, Tij 9 x 11, beta_k 15,
#       T0_k 3 x 7, prefactor 1 = 316; momentum rows 3 x (9 x 8 + 6 + 9) = 261; energy row 3 x 27 + 5 = 86;   663
HAND = {
    ("recon_cell", 0, "weno5"): 99, ("recon_cell", 0, "minmod"): 7,
    ("face_average", 0, "weno5"): 20,
    ("metric_complete_face", 0, "weno5"): 16, ("metric_complete_face", 1, "weno5"): 19, ("metric_complete_face", 2, "weno5"): 19,
    ("admissible", 0, "weno5"): 20, ("prim2con_point", 0, "weno5"): 98,
    ("flux_point", 0, "weno5"): 41, ("flux_point", 1, "weno5"): 41, ("flux_point", 2, "weno5"): 41,
    ("wavespeeds_point", 0, "weno5"): 29, ("wavespeeds_point", 2, "weno5"): 29,
    ("hlle", 0, "weno5"): 72, ("flux_difference", 0, "weno5"): 3, ("derivative", 0, "weno5"): 6,
    ("metric_complete", 0, "weno5"): 30, ("sources_point", 0, "weno5"): 663,
}


@pytest.mark.parametrize("key", sorted(HAND))
def test_piece_counts_match_hand_counts(oracle, key):
    """Pins the counting instance piece by piece against counts made by hand from the formulas (not by calling it)."""
    piece, d, recon = key
    assert sum(oracle.count_piece(piece, d, recon).values()) == HAND[key], key


def hand_total(n, recon):
    """Whole-call operation count assembled from the hand counts: per direction d every line has n_d + 2 reconstructed
    cells (8 variables each), n_d + 1 faces (average, metric completion, 2 x (admissible + state + flux + speeds), HLLE) and
    n_d cells x 8 flux differences; every cell has 30 derivatives, one sources_point and 4 accumulations."""
    rec = HAND[("recon_cell", 0, recon)]
    side = 20 + 98 + 41 + 29
    total = 0
    for d in range(3):
        lines = n[(d + 1) % 3] * n[(d + 2) % 3]
        face = 20 + HAND[("metric_complete_face", d, "weno5")] + 2 * side + 72
        total += lines * ((n[d] + 2) * 8 * rec + (n[d] + 1) * face + n[d] * 8 * 3)
    return total + n[0] * n[1] * n[2] * (30 * 6 + 663 + 4)


@pytest.mark.parametrize("recon", ["weno5", "minmod"])
def test_whole_call_count_equals_hand_assembly(oracle, recon):
    """The counted total of a whole call is EXACTLY the hand counts times the number of times each piece runs
    (WENO5 and minmod have no data-dependent operation), and bench.FLOPS_MODEL's (A, B) are the large-N limit and
    the 1/N coefficient of that assembly."""
    for n in ((12, 9, 7), (16, 16, 16)):
        prob = inputs.general_metric_box(n=n, seed=2)
        _, ops = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma,
                                     variant="count")
        assert sum(ops.values()) == hand_total(n, recon), (n, recon)
    rec = HAND[("recon_cell", 0, recon)]
    a_hand = 24 * rec + (36 + 39 + 39) + 3 * (2 * 188 + 72) + 72 + 847
    b_hand = 3 * 2 * 8 * rec + (36 + 39 + 39) + 3 * (2 * 188 + 72)
    a_model, b_model = bench.FLOPS_MODEL[recon]
    assert abs(a_model - a_hand) <= 1 and abs(b_model - b_hand) <= 2, (a_hand, b_hand)


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
