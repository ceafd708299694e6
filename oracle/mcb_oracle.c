/*
 * mcb_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU oracle for the hot path of Andriati & Gammal,
 * arXiv 2005.13679.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call into this file.  It shares no code,
 * header, table generator or helper with the CUDA library in paper_2005_13679_b200/.
 *
 * What is here, and the passage each function follows:
 *   mcbo_binom_table   N_c(n,m) = binom(n+m-1, m-1), N_c(n,0) = 0     Eq. (7), Eq. (14)
 *   mcbo_rank          Algorithm 1, verbatim (one addition per particle) PAPER.md:132-147
 *   mcbo_unrank        Algorithm 2, verbatim (greedy subtraction)
 *   mcbo_map1          single-jump map  Map1[b][k][l]                    PAPER.md:200-204   (readings A12, A13)
 *   mcbo_map2          double-jump map  Map2[b][(k<=s)][(q<=l)]          PAPER.md:206-224   (reading A15)
 *   mcbo_hc_apply_rows HC_g = sum_b <n^g|H|n^b> C_b for a list of rows g Eq. (3),(4),(12),(13) PAPER.md:49-53,101-107
 *                      H = sum T_kl a+_k a_l + 1/2 sum V_ksql a+_k a+_s a_q a_l (north star; reading A6)
 *   mcbo_rho           rho1[k][l] = <Psi|a+_k a_l|Psi>, rho2[k][s][q][l] = <Psi|a+_k a+_s a_q a_l|Psi>
 *                      Eq. (10),(11) PAPER.md:93-97; index order of App. B PAPER.md:377 (reading A11)
 *
 * The apply is the plain definition: for each output row g the ORDERED sums over (k,l) and
 * (k,s,q,l) are written out, each target index recomputed with the literal O(N) Algorithm 1
 * (the paper's "hashing table + algorithm 1" variant).  No blocking, packing,
 * symmetrisation or reordering.  Arithmetic is C99 double complex (fp64).
 *
 * Pins (tests/test_oracle_*.py): Fig. 1 value 17, nc of the five configs, bijection,
 * independent nested-loop enumeration, brute-force dense H from one-at-a-time ladder operators
 * (oracle/brute.py), App. B rules, Hermiticity, N=1 / M=1 special cases, V=0 spectrum, constant-V and
 * A(x)A closed forms, Lieb-Liniger momentum conservation and ground-state energy vs exact
 * diagonalisation and the Bethe-ansatz bound.  Parity at the five full-size configs has no pin
 * outside this oracle beyond those invariants ("parity unpinned beyond the oracle" at full size).
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex zc;

#define MCBO_MAXM 64

/* ---- Eq. (7), (14): N_c(n,m) = binom(n+m-1, m-1); N_c(n,0) = 0; hence N_c(0,m>=1) = 1 ---------------- */
/* out is row-major [n][m], (N+1) x (M+1).  Pascal: N_c(n,m) = N_c(n-1,m) + N_c(n,m-1).  Returns 0, or -1
 * if any entry would exceed 2^62 (the caller then must not use the table). */
int mcbo_binom_table(int N, int M, long long *out)
{
    const long long LIM = (long long)1 << 62;
    int W = M + 1;
    for (int n = 0; n <= N; ++n) out[n * W + 0] = 0;
    for (int m = 1; m <= M; ++m) out[0 * W + m] = 1;
    for (int n = 1; n <= N; ++n) {
        /* N_c(n,1) = binom(n,0) = 1: one orbital, one configuration.  (N_c(n,0) = 0 is the cost
         * convention of Eq. (14), not a Pascal seed.) */
        out[n * W + 1] = 1;
        for (int m = 2; m <= M; ++m) {
            long long a = out[(n - 1) * W + m];   /* binom(n+m-2, m-1) */
            long long b = out[n * W + (m - 1)];   /* binom(n+m-2, m-2) */
            if (a > LIM - b) return -1;
            out[n * W + m] = a + b;
        }
    }
    return 0;
}

/* helper: table lookup */
static inline long long NC(const long long *tab, int M, int n, int m) { return tab[n * (M + 1) + m]; }

/* ---- Algorithm 1, verbatim ------------------------------------------------------- */
long long mcbo_rank(int N, int M, const long long *tab, const int *n)
{
    long long k = 0;
    int s = N;
    for (int m = M - 1; m >= 1; --m) {
        int j = n[m];
        while (j > 0) {
            k = k + NC(tab, M, s, m);
            s = s - 1;
            j = j - 1;
        }
    }
    return k;
}

/* ---- Algorithm 2, verbatim; accepts beta = 0 (reading A2) ------------------------- */
void mcbo_unrank(int N, int M, const long long *tab, long long beta, int *n)
{
    for (int i = 0; i <= M - 1; ++i) n[i] = 0;
    long long k = beta;
    int m = M - 1;
    int s = N;
    while (k > 0) {
        while (k - NC(tab, M, s, m) < 0) m = m - 1;
        k = k - NC(tab, M, s, m);
        n[m] = n[m] + 1;
        s = s - 1;
    }
    if (s > 0) n[0] = n[0] + s;
}

void mcbo_rank_batch(int N, int M, const int *occ, long long batch, long long *idx)
{
    long long *tab = (long long *)malloc(sizeof(long long) * (size_t)(N + 1) * (M + 1));
    mcbo_binom_table(N, M, tab);
    for (long long b = 0; b < batch; ++b) idx[b] = mcbo_rank(N, M, tab, occ + b * M);
    free(tab);
}

void mcbo_unrank_batch(int N, int M, const long long *idx, long long batch, int *occ)
{
    long long *tab = (long long *)malloc(sizeof(long long) * (size_t)(N + 1) * (M + 1));
    mcbo_binom_table(N, M, tab);
    for (long long b = 0; b < batch; ++b) mcbo_unrank(N, M, tab, idx[b], occ + b * M);
    free(tab);
}

/* ---- Single-jump map: Map1[b][k][l] = index of n^(b) - e_k + e_l if n_k >= 1, else -1
 *      (A12); the diagonal k == l is b itself if n_k >= 1, else -1 (A13).  out: [count][M][M] ---------- */
void mcbo_map1(int N, int M, long long b0, long long count, long long *out)
{
    long long *tab = (long long *)malloc(sizeof(long long) * (size_t)(N + 1) * (M + 1));
    mcbo_binom_table(N, M, tab);
    int n[MCBO_MAXM];
    for (long long i = 0; i < count; ++i) {
        mcbo_unrank(N, M, tab, b0 + i, n);
        for (int k = 0; k < M; ++k)
            for (int l = 0; l < M; ++l) {
                long long v = -1;
                if (n[k] >= 1) {
                    n[k] -= 1; n[l] += 1;
                    v = mcbo_rank(N, M, tab, n);
                    n[l] -= 1; n[k] += 1;
                }
                out[(i * M + k) * M + l] = v;
            }
    }
    free(tab);
}

/* ---- Double-jump map (reading A15): for every unordered removal pair k <= s that is
 *      allowed (n_k >= 1, n_s >= 1, and n_k >= 2 when k == s) and every unordered insertion pair q <= l,
 *      the index of n - e_k - e_s + e_q + e_l; -1 where the removal is not allowed.
 *      Pair order: (0,0),(0,1),..,(0,M-1),(1,1),..,(M-1,M-1).  out: [count][P][P], P = M(M+1)/2 --------- */
void mcbo_map2(int N, int M, long long b0, long long count, long long *out)
{
    long long *tab = (long long *)malloc(sizeof(long long) * (size_t)(N + 1) * (M + 1));
    mcbo_binom_table(N, M, tab);
    int P = M * (M + 1) / 2;
    int n[MCBO_MAXM];
    for (long long i = 0; i < count; ++i) {
        mcbo_unrank(N, M, tab, b0 + i, n);
        int a = 0;
        for (int k = 0; k < M; ++k)
            for (int s = k; s < M; ++s, ++a) {
                int ok = (k == s) ? (n[k] >= 2) : (n[k] >= 1 && n[s] >= 1);
                int c = 0;
                for (int q = 0; q < M; ++q)
                    for (int l = q; l < M; ++l, ++c) {
                        long long v = -1;
                        if (ok) {
                            n[k] -= 1; n[s] -= 1; n[q] += 1; n[l] += 1;
                            v = mcbo_rank(N, M, tab, n);
                            n[l] -= 1; n[q] -= 1; n[s] += 1; n[k] += 1;
                        }
                        out[(i * P + a) * P + c] = v;
                    }
            }
    }
    free(tab);
}

/* ---- H.C for a list of output rows (Eq. 12-13; three-step recipe PAPER.md:176) -------
 *  H = sum_{k,l} T[k][l] a+_k a_l  +  1/2 sum_{k,s,q,l} V[k][s][q][l] a+_k a+_s a_q a_l.
 *  <n^g| a+_k a_l |n^b> != 0 iff n^b = n^g - e_k + e_l, amplitude sqrt(n^b_l) sqrt(n^g_k)
 *      = sqrt(n_k (n_l + 1))  (k != l),  n_k  (k == l)            with n = n^g       (Eq. 1, 5 PAPER.md:39,61)
 *  <n^g| a+_k a+_s a_q a_l |n^b> != 0 iff n^b = m + e_q + e_l, m = n^g - e_k - e_s >= 0, amplitude
 *      sqrt(n_k (n_s - [k==s])) * sqrt((m_q + 1)(m_l + 1 + [q==l])).
 *  The integer radicand is < 2^53, so sqrt() of it is the correctly rounded value of the exact amplitude.
 *  rows == NULL means rows 0..nrows-1.  nthreads <= 0: OpenMP default.  Returns threads used. */
int mcbo_hc_apply_rows(int N, int M, const zc *T, const zc *V, const zc *C,
                       const long long *rows, long long nrows, zc *out, int nthreads)
{
    long long *tab = (long long *)malloc(sizeof(long long) * (size_t)(N + 1) * (M + 1));
    mcbo_binom_table(N, M, tab);
    int used = 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#pragma omp parallel
    {
#pragma omp single
        used = omp_get_num_threads();
    }
#pragma omp parallel for schedule(dynamic, 16)
#endif
    for (long long r = 0; r < nrows; ++r) {
        long long g = rows ? rows[r] : r;
        int n[MCBO_MAXM];
        mcbo_unrank(N, M, tab, g, n);
        zc acc = 0.0;
        /* one-body */
        for (int k = 0; k < M; ++k) {
            if (n[k] < 1) continue;
            for (int l = 0; l < M; ++l) {
                if (l == k) {
                    acc += T[k * M + k] * (double)n[k] * C[g];
                } else {
                    double amp = sqrt((double)((long long)n[k] * (n[l] + 1)));
                    n[k] -= 1; n[l] += 1;
                    long long b = mcbo_rank(N, M, tab, n);
                    n[l] -= 1; n[k] += 1;
                    acc += T[k * M + l] * amp * C[b];
                }
            }
        }
        /* two-body, ordered quadruple sum */
        for (int k = 0; k < M; ++k)
            for (int s = 0; s < M; ++s) {
                long long f1 = (long long)n[k] * (n[s] - (k == s ? 1 : 0));
                if (f1 <= 0) continue;
                n[k] -= 1; n[s] -= 1;               /* n is now m */
                for (int q = 0; q < M; ++q)
                    for (int l = 0; l < M; ++l) {
                        long long f2 = (long long)(n[q] + 1) * (n[l] + 1 + (q == l ? 1 : 0));
                        double amp = sqrt((double)(f1 * f2));
                        n[q] += 1; n[l] += 1;
                        long long b = mcbo_rank(N, M, tab, n);
                        n[l] -= 1; n[q] -= 1;
                        acc += 0.5 * V[((k * M + s) * M + q) * M + l] * amp * C[b];
                    }
                n[s] += 1; n[k] += 1;
            }
        out[r] = acc;
    }
    free(tab);
    return used;
}

/* ---- Eq. (10), (11): one- and two-body density matrices ---------------------------------------------------
 *  rho1[k*M+l] = sum_{g,b} conj(C_g) C_b <n^g| a+_k a_l |n^b>,
 *  rho2[((k*M+s)*M+q)*M+l] = sum_{g,b} conj(C_g) C_b <n^g| a+_k a+_s a_q a_l |n^b>   (App. B labels rho_ksql),
 *  written out as the double sum: for every bra g and every ordered index tuple the single ket b with a non-zero
 *  element is found by the literal Algorithm 1, amplitudes as in mcbo_hc_apply_rows (ladder algebra, Eq. 1, 5).
 *  Serial, one accumulation order.  With these conventions <Psi|H|Psi> = sum T_kl rho1_kl + 1/2 sum V_ksql rho2_ksql. */
void mcbo_rho(int N, int M, const zc *C, zc *rho1, zc *rho2)
{
    long long *tab = (long long *)malloc(sizeof(long long) * (size_t)(N + 1) * (M + 1));
    mcbo_binom_table(N, M, tab);
    const long long nc = NC(tab, M, N, M);
    for (int i = 0; i < M * M; ++i) rho1[i] = 0.0;
    for (long long i = 0; i < (long long)M * M * M * M; ++i) rho2[i] = 0.0;
    for (long long g = 0; g < nc; ++g) {
        int n[MCBO_MAXM];
        mcbo_unrank(N, M, tab, g, n);
        const zc cg = conj(C[g]);
        for (int k = 0; k < M; ++k) {
            if (n[k] < 1) continue;
            for (int l = 0; l < M; ++l) {
                if (l == k) {
                    rho1[k * M + k] += cg * (double)n[k] * C[g];
                } else {
                    double amp = sqrt((double)((long long)n[k] * (n[l] + 1)));
                    n[k] -= 1; n[l] += 1;
                    long long b = mcbo_rank(N, M, tab, n);
                    n[l] -= 1; n[k] += 1;
                    rho1[k * M + l] += cg * amp * C[b];
                }
            }
        }
        for (int k = 0; k < M; ++k)
            for (int s = 0; s < M; ++s) {
                long long f1 = (long long)n[k] * (n[s] - (k == s ? 1 : 0));
                if (f1 <= 0) continue;
                n[k] -= 1; n[s] -= 1;               /* n is now m */
                for (int q = 0; q < M; ++q)
                    for (int l = 0; l < M; ++l) {
                        long long f2 = (long long)(n[q] + 1) * (n[l] + 1 + (q == l ? 1 : 0));
                        double amp = sqrt((double)(f1 * f2));
                        n[q] += 1; n[l] += 1;
                        long long b = mcbo_rank(N, M, tab, n);
                        n[l] -= 1; n[q] -= 1;
                        rho2[((k * M + s) * M + q) * M + l] += cg * amp * C[b];
                    }
                n[s] += 1; n[k] += 1;
            }
    }
    free(tab);
}

int mcbo_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
