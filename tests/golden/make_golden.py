"""Writes the text fixtures under tests/golden/.  Calls only ``oracle/`` and the shared input
generators (``tdma_inputs``) -- never the CUDA path.

  second_difference_inverse.txt  closed form, no solver involved: the inverse of the n x n
        second-difference matrix tridiag(-1, 2, -1) is min(i,j) (n+1-max(i,j)) / (n+1)
        (textbook Green's function of the discrete Dirichlet Laplacian); stored as the exact
        integer numerators over (n+1).
  cfg1_oracle_lines.txt          oracle solution (fp64 Thomas) of four lines of BASELINE cfg 1
        (64^3, seed 0), as hex floats; a regression anchor for the oracle and the generators
        and a fixed target for the GPU parity test.

Run from the repo root:  python tests/golden/make_golden.py
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

LINES = [(0, 0), (17, 3), (63, 63), (5, 40)]          # (i, k)


def main():
    n = 6
    with open(os.path.join(HERE, "second_difference_inverse.txt"), "w") as f:
        f.write("# numerators of (tridiag(-1,2,-1))^-1 over (n+1): min(i,j)*(n+1-max(i,j)), i,j=1..n\n")
        f.write("# closed form (discrete Dirichlet Green's function); first row: n\n")
        f.write("%d\n" % n)
        for i in range(1, n + 1):
            f.write(" ".join(str(min(i, j) * (n + 1 - max(i, j))) for j in range(1, n + 1)) + "\n")

    import oracle
    import tdma_inputs
    w = tdma_inputs.make_workload("cfg1_tiny")
    x = oracle.solve_y(w.a.numpy(), w.b.numpy(), w.c.numpy(), w.d.numpy())
    with open(os.path.join(HERE, "cfg1_oracle_lines.txt"), "w") as f:
        f.write("# oracle.solve_y (fp64 Thomas, PAPER.md:11) on BASELINE cfg 1 (64x64x64, seed 0)\n")
        f.write("# one line per row: i k x_0 ... x_63 as C99 hex floats\n")
        for (i, k) in LINES:
            f.write("%d %d " % (i, k) + " ".join(float(v).hex() for v in x[k, :, i]) + "\n")


if __name__ == "__main__":
    main()
