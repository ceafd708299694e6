"""Seeded synthetic input generators for the five BASELINE.json configs.

This module is shared by the tests, bench.py and __graft_entry__.smoke(): it
hands the *same* numpy arrays to the CPU oracle (oracle/) and to the CUDA
library (paper_2005_13679_b200/).  It holds none of the method's arithmetic:
no binomial table, no hashing, no matrix elements -- only the random / analytic
*inputs* T, V, C and index batches, following the recipe in SURVEY.md 8(d) and
DESIGN.md ("Input recipe").

The paper measures on no public dataset: its workload is "randomly generating
the components of the vector C, normalizing it to one" over an
M=3 / large-N sweep and an N=5 / large-M sweep plus
Lieb-Liniger plane waves.  The configs below keep those shapes
at nc ~ 1e7 (BASELINE.json:configs).
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

SEED_BASE = 200513679


@dataclass(frozen=True)
class Config:
    cfg: int
    name: str
    N: int
    M: int
    nc: int          # the value BASELINE.json prints (checked against the table in tests)
    kind: str        # "dense" | "ll"


CONFIGS = (
    Config(0, "tiny", 10, 5, 1001, "dense"),
    Config(1, "lieb_liniger", 100, 5, 4598126, "ll"),
    Config(2, "many_particles_few_orbitals", 400, 4, 10827401, "dense"),
    Config(3, "balanced", 20, 10, 10015005, "dense"),
    Config(4, "orbital_heavy", 15, 12, 7726160, "dense"),
)


def seed_for(cfg: int, stream: int = 0) -> int:
    return SEED_BASE + cfg + 1000 * stream


def _cnormal(rng: np.random.Generator, shape) -> np.ndarray:
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def random_hermitian_T(M: int, rng: np.random.Generator) -> np.ndarray:
    """T = (A + A^H)/2, A_kl = N(0,1) + i N(0,1).  complex128 [M, M]."""
    A = _cnormal(rng, (M, M))
    return np.ascontiguousarray((A + A.conj().T) / 2)


def random_symmetric_V(M: int, rng: np.random.Generator) -> np.ndarray:
    """Random complex V[k,s,q,l] with V_ksql = V_skql = V_kslq and V_ksql = conj(V_lqsk).

    (BASELINE.json configs[0].)  complex128 [M, M, M, M].
    """
    G = _cnormal(rng, (M, M, M, M))
    V = (G + G.transpose(1, 0, 2, 3) + G.transpose(0, 1, 3, 2) + G.transpose(1, 0, 3, 2)) / 4
    # V_ksql <- (V_ksql + conj(V_lqsk))/2 : axes (k,s,q,l) <- (l,q,s,k)
    V = (V + V.conj().transpose(3, 2, 1, 0)) / 2
    return np.ascontiguousarray(V)


def random_general_V(M: int, rng: np.random.Generator) -> np.ndarray:
    """Completely unsymmetric complex V (the ABI accepts any M^4 tensor)."""
    return np.ascontiguousarray(_cnormal(rng, (M, M, M, M)))


def lieb_liniger_TV(M: int, g: float = 10.0, L: float = 1.0):
    """Plane-wave orbitals on a ring: orbital j <-> momentum p_j = j - (M-1)/2 (M odd).

    T_kk = (2 pi p_k / L)^2 / 2 (hbar = m = 1), T off-diagonal 0;
    V_ksql = g/L if p_k + p_s == p_q + p_l else 0.   (BASELINE.json configs[1])
    """
    if M % 2 != 1:
        raise ValueError("Lieb-Liniger workload wants an odd number of plane waves")
    p = np.arange(M) - (M - 1) // 2
    T = np.zeros((M, M), dtype=np.complex128)
    T[np.arange(M), np.arange(M)] = 0.5 * (2.0 * math.pi * p / L) ** 2
    k, s, q, l = np.meshgrid(p, p, p, p, indexing="ij")
    V = np.where(k + s == q + l, g / L, 0.0).astype(np.complex128)
    return np.ascontiguousarray(T), np.ascontiguousarray(V), p


def bose_hubbard_TV(M: int, J: float = 1.0, U: float = 4.0, ring: bool = True):
    """Bose-Hubbard specialisation the paper names: M sites, nearest-neighbour hopping
    T_kl = -J for |k - l| = 1 (and the ring bond 0 <-> M-1), on-site interaction V_kkkk = U
    (H = -J sum <kl> a+_k a_l + U/2 sum n_k (n_k - 1)); everything else zero."""
    T = np.zeros((M, M), dtype=np.complex128)
    for k in range(M - 1):
        T[k, k + 1] = T[k + 1, k] = -J
    if ring and M > 2:
        T[0, M - 1] = T[M - 1, 0] = -J
    V = np.zeros((M, M, M, M), dtype=np.complex128)
    for k in range(M):
        V[k, k, k, k] = U
    return T, V


def random_normalised_C(nc: int, rng: np.random.Generator) -> np.ndarray:
    """C = randn + i randn, L2-normalised.  complex128 [nc]."""
    C = np.empty(nc, dtype=np.complex128)
    C.real = rng.standard_normal(nc)
    C.imag = rng.standard_normal(nc)
    C /= np.linalg.norm(C)
    return C


def make_inputs(cfg: int, n_vectors: int = 1):
    """(Config, T, V, [C_0 .. C_{n_vectors-1}]) for one of the five configs, seeded."""
    c = CONFIGS[cfg]
    rng = np.random.default_rng(seed_for(cfg))
    if c.kind == "ll":
        T, V, _ = lieb_liniger_TV(c.M)
    else:
        T = random_hermitian_T(c.M, rng)
        V = random_symmetric_V(c.M, rng)
    Cs = [random_normalised_C(c.nc, rng) for _ in range(n_vectors)]
    return c, T, V, Cs


def make_small_inputs(N: int, M: int, nc: int, seed: int, kind: str = "dense", general_V: bool = False):
    """Inputs for an arbitrary small (N, M); nc is supplied by the caller (no arithmetic here)."""
    rng = np.random.default_rng(seed)
    if kind == "ll":
        T, V, _ = lieb_liniger_TV(M)
    elif kind == "bh":
        T, V = bose_hubbard_TV(M)
    else:
        T = random_hermitian_T(M, rng)
        V = random_general_V(M, rng) if general_V else random_symmetric_V(M, rng)
    C = random_normalised_C(nc, rng)
    return T, V, C


def index_batch(nc: int, batch: int, seed: int) -> np.ndarray:
    """Seeded random batch of indices in [0, nc), int32."""
    rng = np.random.default_rng(seed)
    return rng.integers(0, nc, size=batch, dtype=np.int64).astype(np.int32)


def sample_rows(nc: int, n_head: int, n_random: int, seed: int) -> np.ndarray:
    """Row subset used for bounded oracle runs: first n_head rows, last n_head rows and
    n_random seeded random rows (rows of H.C are independent).  Sorted unique int64."""
    rng = np.random.default_rng(seed)
    head = np.arange(min(n_head, nc), dtype=np.int64)
    tail = np.arange(max(nc - n_head, 0), nc, dtype=np.int64)
    rnd = rng.integers(0, nc, size=n_random, dtype=np.int64)
    return np.unique(np.concatenate([head, tail, rnd]))
