"""oracle.lanczos -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain numpy Lanczos tridiagonalisation with full re-orthogonalisation, every H.v through the CPU
oracle's hc_apply (oracle/mcb_oracle.c).  Written out step by step in the usual notation:

    v_0 = v0/|v0|;  for j = 0..k-1:  w = H v_j;  c_i = <v_i|w> (i <= j), alpha_j = Re c_j;  w -= sum c_i v_i  (twice);
                                     beta_j = |w|;  v_{j+1} = w / beta_j.

Pins (tests/test_oracle_lanczos.py): with k = nc the tridiagonal matrix has the spectrum of the brute-force dense H;
the basis is orthonormal; the Lieb-Liniger ground-state energy equals exact diagonalisation and lies above the
Bethe-ansatz value.  Shares no code with paper_2005_13679_b200.
"""
from __future__ import annotations

import numpy as np

from . import hc_apply


def lanczos(N: int, M: int, T, V, v0, kmax: int, breakdown: float = 1e-12):
    """(alpha [k], beta [k], basis [k+1 or k, nc]) -- k <= kmax steps (stops at an invariant subspace)."""
    v0 = np.asarray(v0, dtype=np.complex128)
    basis = [v0 / np.linalg.norm(v0)]
    alpha, beta = [], []
    for j in range(kmax):
        w, _ = hc_apply(N, M, T, V, basis[j])
        a = 0.0
        for _ in range(2):
            c = [np.vdot(v, w) for v in basis]
            for ci, v in zip(c, basis):
                w = w - ci * v
            a += c[j].real
        alpha.append(a)
        b = float(np.linalg.norm(w))
        beta.append(b)
        if j + 1 == kmax or b <= breakdown * max(1.0, abs(alpha[0])):
            break
        basis.append(w / b)
    return np.array(alpha), np.array(beta), np.array(basis)


def ritz_values(alpha, beta):
    """Eigenvalues of tridiag(alpha, beta[:-1]) (the host-side solve of the paper, here by numpy's dense eigvalsh)."""
    k = len(alpha)
    Tm = np.diag(np.asarray(alpha, dtype=np.float64))
    for j in range(k - 1):
        Tm[j, j + 1] = Tm[j + 1, j] = beta[j]
    return np.linalg.eigvalsh(Tm)
