"""oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes wrapper around oracle/mcb_oracle.c (plain C, fp64, OpenMP only for the timed all-cores leg).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
It never imports paper_2005_13679_b200 and shares no code with it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mcb_oracle.c")
_LIB = os.path.join(_HERE, "libmcb_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -shared; rebuilt when the source is newer than the library."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        ll, i, p = ctypes.c_longlong, ctypes.c_int, ctypes.c_void_p
        L.mcbo_binom_table.argtypes = [i, i, p]
        L.mcbo_binom_table.restype = i
        L.mcbo_rank_batch.argtypes = [i, i, p, ll, p]
        L.mcbo_unrank_batch.argtypes = [i, i, p, ll, p]
        L.mcbo_map1.argtypes = [i, i, ll, ll, p]
        L.mcbo_map2.argtypes = [i, i, ll, ll, p]
        L.mcbo_hc_apply_rows.argtypes = [i, i, p, p, p, p, ll, p, i]
        L.mcbo_hc_apply_rows.restype = i
        L.mcbo_max_threads.restype = i
        L.mcbo_rho.argtypes = [i, i, p, p, p]
        L.mcbo_rho.restype = None
        _lib = L
    return _lib


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def binom_table(N: int, M: int) -> np.ndarray:
    """int64 [(N+1), (M+1)]: N_c(n, m) = binom(n+m-1, m-1), N_c(n, 0) = 0 (Eq. 7, 14)."""
    out = np.zeros((N + 1, M + 1), dtype=np.int64)
    rc = lib().mcbo_binom_table(N, M, _ptr(out))
    if rc != 0:
        raise OverflowError("binomial table overflows int64")
    return out


def nc(N: int, M: int) -> int:
    return int(binom_table(N, M)[N, M])


def rank(N: int, M: int, occ: np.ndarray) -> np.ndarray:
    """Algorithm 1 on each row of occ [batch, M] -> int64 [batch]."""
    occ = np.ascontiguousarray(occ, dtype=np.int32).reshape(-1, M)
    idx = np.empty(occ.shape[0], dtype=np.int64)
    lib().mcbo_rank_batch(N, M, _ptr(occ), occ.shape[0], _ptr(idx))
    return idx


def unrank(N: int, M: int, idx: np.ndarray) -> np.ndarray:
    """Algorithm 2 on each index -> int32 [batch, M]."""
    idx = np.ascontiguousarray(idx, dtype=np.int64).reshape(-1)
    occ = np.empty((idx.shape[0], M), dtype=np.int32)
    lib().mcbo_unrank_batch(N, M, _ptr(idx), idx.shape[0], _ptr(occ))
    return occ


def map1(N: int, M: int, b0: int, count: int) -> np.ndarray:
    """int64 [count, M, M]; -1 = forbidden (n_k = 0)."""
    out = np.empty((count, M, M), dtype=np.int64)
    lib().mcbo_map1(N, M, b0, count, _ptr(out))
    return out


def map2(N: int, M: int, b0: int, count: int) -> np.ndarray:
    """int64 [count, P, P], P = M(M+1)/2, pairs ordered (0,0),(0,1)..(M-1,M-1); -1 = removal not allowed."""
    P = M * (M + 1) // 2
    out = np.empty((count, P, P), dtype=np.int64)
    lib().mcbo_map2(N, M, b0, count, _ptr(out))
    return out


def map2_compact(N: int, M: int, b0: int, count: int):
    """The paper's COMPACT double-jump table (Fig. 3) for lines b0 .. b0 + count - 1, written out as the
    text says: "for every non-empty IPS k we search for s >= k non-empty as well, and whenever we find such numbers" the
    line gets one stride with the configurations reached by putting the two particles back -- here the P = M(M+1)/2
    unordered replacements (q <= l) in pair order (the paper's M^2 stride lists each q != l target twice).  Every target by
    the literal Algorithm 1 (rank).  Returns (offsets int64 [count + 1], relative to line b0; strides int64 [n, P];
    pairs int64 [n, 2], the removal (k, s) of every stride)."""
    P = M * (M + 1) // 2
    occ = unrank(N, M, np.arange(b0, b0 + count, dtype=np.int64))
    offsets = [0]
    removed, pairs = [], []
    for row in occ:
        row = row.astype(np.int64)
        cnt = 0
        for k in range(M):
            if row[k] < 1:
                continue
            for s in range(k, M):
                if (s == k and row[k] < 2) or (s != k and row[s] < 1):
                    continue
                m = row.copy()
                m[k] -= 1
                m[s] -= 1
                removed.append(m)
                pairs.append((k, s))
                cnt += 1
        offsets.append(offsets[-1] + cnt)
    n = len(removed)
    strides = np.empty((n, P), dtype=np.int64)
    if n:
        base = np.asarray(removed, dtype=np.int64)
        c = 0
        for q in range(M):
            for l in range(q, M):
                tgt = base.copy()
                tgt[:, q] += 1
                tgt[:, l] += 1
                strides[:, c] = rank(N, M, tgt)
                c += 1
    return np.asarray(offsets, dtype=np.int64), strides, np.asarray(pairs, dtype=np.int64).reshape(n, 2)


def hc_apply(N: int, M: int, T: np.ndarray, V: np.ndarray, C: np.ndarray,
             rows: np.ndarray | None = None, nthreads: int = 0):
    """HC restricted to `rows` (all rows if None).  Returns (complex128 [nrows], threads used)."""
    T = np.ascontiguousarray(T, dtype=np.complex128).reshape(M, M)
    V = np.ascontiguousarray(V, dtype=np.complex128).reshape(M, M, M, M)
    C = np.ascontiguousarray(C, dtype=np.complex128).reshape(-1)
    if rows is None:
        nrows = C.shape[0]
        rp = None
    else:
        rows = np.ascontiguousarray(rows, dtype=np.int64).reshape(-1)
        nrows = rows.shape[0]
        rp = _ptr(rows)
    out = np.empty(nrows, dtype=np.complex128)
    used = lib().mcbo_hc_apply_rows(N, M, _ptr(T), _ptr(V), _ptr(C), rp, nrows, _ptr(out), nthreads)
    return out, used


def rho(N: int, M: int, C: np.ndarray):
    """(rho1 [M,M], rho2 [M,M,M,M]) complex128: <a+_k a_l>, <a+_k a+_s a_q a_l> (Eq. 10, 11; App. B index order)."""
    C = np.ascontiguousarray(C, dtype=np.complex128).reshape(-1)
    r1 = np.empty((M, M), dtype=np.complex128)
    r2 = np.empty((M, M, M, M), dtype=np.complex128)
    lib().mcbo_rho(N, M, _ptr(C), _ptr(r1), _ptr(r2))
    return r1, r2


def max_threads() -> int:
    return int(lib().mcbo_max_threads())
