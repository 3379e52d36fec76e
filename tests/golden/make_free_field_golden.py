"""Writes tests/golden/free_field_eigenvalues.txt from the closed form alone (no oracle, no CUDA).

Free field (U = 1, F = 0) in Eq. 1: for psi(x) = exp(i p x) chi with
p_mu = 2 pi (n_mu + 1/2 [bc_mu = -1]) / L_mu the operator acts as the 12x12 matrix
M(p) = (1 - 2 kappa sum_mu cos p_mu) + 2 i kappa sum_mu gamma_mu sin p_mu, whose eigenvalues are
    1 - 2 kappa sum_mu cos p_mu  +-  2 i kappa sqrt(sum_mu sin^2 p_mu),   each six-fold
for ANY Hermitian gamma matrices obeying {gamma_mu, gamma_nu} = 2 delta.  The paper prints no
worked numbers; these are the values its Eq. 1 fixes.
Columns: Lx Ly Lz Lt  nx ny nz nt  bcx bcy bcz bct  kappa  Re(lambda)  |Im(lambda)|
"""
import math
import os

CASES = [
    ((4, 4, 4, 4), (1, 2, 0, 1), (1, 1, 1, -1), 0.13),
    ((4, 4, 4, 4), (0, 0, 0, 0), (1, 1, 1, 1), 0.125),
    ((6, 4, 2, 8), (5, 1, 1, 3), (1, 1, 1, -1), 0.1372),
    ((4, 2, 4, 6), (3, 0, 2, 4), (-1, -1, 1, -1), 0.12),
]

here = os.path.dirname(os.path.abspath(__file__))
with open(os.path.join(here, "free_field_eigenvalues.txt"), "w") as f:
    f.write("# closed-form free-field eigenvalues of Eq. 1 (PAPER.md:47); written by make_free_field_golden.py\n")
    f.write("# Lx Ly Lz Lt  nx ny nz nt  bcx bcy bcz bct  kappa  Re(lambda)  |Im(lambda)|\n")
    for dims, n, bc, kappa in CASES:
        p = [2 * math.pi * (n[m] + (0.5 if bc[m] == -1 else 0.0)) / dims[m] for m in range(4)]
        re = 1 - 2 * kappa * sum(math.cos(q) for q in p)
        im = 2 * kappa * math.sqrt(sum(math.sin(q) ** 2 for q in p))
        f.write(" ".join(str(v) for v in dims + n + bc) + f" {kappa} {re:.9f} {im:.9f}\n")
