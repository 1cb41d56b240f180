"""Writes the algorithmic operation count that bench.py's roofline uses (FLOPS_MODEL): TEST/BENCH INFRASTRUCTURE.

    python -m oracle.count_flops

Runs the oracle's COUNTING instance (every +, -, *, /, sqrt of the straightforward formulation counted as one
operation, an FMA would be two; every face evaluated once) on cubic general-metric boxes
of N = 16, 32, 48 interior cells and fits  flops per cell-update = A + B / N  (the 1/N term is the extra plane of
faces per direction).  Calls only oracle/ and the seeded input generators; prints the table and the fitted
(A, B) per reconstruction, which are the numbers stored in bench.FLOPS_MODEL (tests/test_bench_model.py checks
that they still agree with the oracle)."""
import numpy as np

from oracle import oracle as orc
from paper_2210_17509_b200 import inputs


def main():
    orc.lib()
    sizes = (16, 32, 48)
    for recon in ("weno5", "minmod", "mc"):
        per_cell = []
        for n in sizes:
            prob = inputs.general_metric_box(n=(n, n, n), seed=2)
            _, ops = orc.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma,
                                      variant="count")
            per_cell.append(sum(ops.values()) / prob.cells)
        a_mat = np.stack([np.ones(len(sizes)), 1.0 / np.array(sizes, dtype=float)], axis=1)
        (a, b), *_ = np.linalg.lstsq(a_mat, np.array(per_cell), rcond=None)
        print(f"{recon:7s} " + "  ".join(f"N={n}: {v:9.2f}" for n, v in zip(sizes, per_cell)) +
              f"   fit A = {a:8.1f}, B = {b:8.1f}   -> {a + b / 256:8.1f} flops per cell-update at 256^3")


if __name__ == "__main__":
    main()
