"""oracle.extended -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

The plain definition of H.C (Eq. 12-13; O6 of SURVEY.md 8(c)) for TWO orbitals, evaluated in extended
precision (numpy longdouble: the x87 80-bit format on x86-64, 64-bit mantissa), so that the fp64 rounding of the fp64
oracle itself can be measured where the north-star tolerance 1e-12 * ||T,V||max * ||C||_1 comes within a few ulp of the
result (N = 2000: amplitudes up to N^2).

For M = 2 the order of Eq. (14) makes the index of |n_0, n_1> equal to n_1 (pinned against Algorithm 1 in
tests/test_oracle_apply.py), so no hashing is needed here and nothing is shared with oracle/mcb_oracle.c beyond the formula:

    HC_g = sum_k T_kk n_k C_g + sum_{k != l} T_kl sqrt(n_k (n_l + 1)) C[g_k^l]
         + 1/2 sum_{k,s,q,l} V_ksql sqrt(n_k (n_s - d_ks)) sqrt((m_q + 1)(m_l + 1 + d_ql)) C[index(m + e_q + e_l)],  m = n - e_k - e_s >= 0.
"""
from __future__ import annotations

import numpy as np


def hc_apply_m2_longdouble(N: int, T, V, C) -> np.ndarray:
    """clongdouble vector HC = H.C for M = 2 (nc = N + 1), every operation in extended precision."""
    ld, cld = np.longdouble, np.clongdouble
    T = np.asarray(T, dtype=np.complex128).astype(cld)
    V = np.asarray(V, dtype=np.complex128).astype(cld).reshape(2, 2, 2, 2)
    C = np.asarray(C, dtype=np.complex128).astype(cld)
    nc = N + 1
    assert C.shape == (nc,)
    b = np.arange(nc, dtype=np.int64)                 # index = n_1
    n = [N - b, b]                                    # occupations of orbital 0, 1 per configuration
    acc = np.zeros(nc, dtype=cld)

    def gather(idx, ok):
        out = np.zeros(nc, dtype=cld)
        out[ok] = C[idx[ok]]
        return out

    for k in range(2):
        acc += T[k, k] * n[k].astype(ld) * C
        l = 1 - k
        ok = n[k] >= 1
        tgt = b + (1 if l == 1 else -1)               # one particle k -> l changes n_1 by +-1
        amp = np.sqrt((n[k] * (n[l] + 1)).astype(ld))
        acc += T[k, l] * np.where(ok, amp, ld(0)) * gather(tgt, ok)
    half = ld(1) / ld(2)
    for k in range(2):
        for s in range(2):
            f1 = n[k] * (n[s] - (1 if k == s else 0))
            ok = f1 >= 1
            m = [n[0] - (k == 0) - (s == 0), n[1] - (k == 1) - (s == 1)]
            for q in range(2):
                for l in range(2):
                    f2 = (m[q] + 1) * (m[l] + 1 + (1 if q == l else 0))
                    tgt = m[1] + (q == 1) + (l == 1)
                    amp = np.sqrt(np.where(ok, f1 * f2, 0).astype(ld))
                    acc += half * V[k, s, q, l] * amp * gather(tgt, ok)
    return acc
