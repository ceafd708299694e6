// mcb_device.cuh -- device helpers shared by the libmcb kernels: index arithmetic on prefix sums.
//
// Notation: n = (n_0..n_{M-1}) occupation vector, S_j = n_0 + .. + n_j (S_{M-1} = N),
// G[j][s] = binom(s + j, j + 1).  The index of Algorithm 1 / Eq. (14) is
//     index(n) = nc - 1 - sum_{j=0}^{M-2} G[j][S_j].
// Proof sketch: Algorithm 1 adds, for the particles in orbital m, N_c(s, m) for s = S_m, S_m - 1, .., S_{m-1} + 1,
// which telescopes (hockey stick) to N_c(S_m, m+1) - N_c(S_{m-1}, m+1); summing over m and using
// N_c(N, M) - 1 = sum_m [..] for the last configuration gives the complement form above.
#pragma once
#include "mcb_internal.cuh"

// compile-time M (MT >= 1) or run-time M (MT == 0, arrays sized MCB_MAX_M and kept in local memory)
template <int MT> struct MTraits { static constexpr int CAP = MT ? MT : MCB_MAX_M; };

__device__ __forceinline__ int mcb_ldG(const int* __restrict__ G, int ldg, int j, int s) { return __ldg(G + j * ldg + s); }

// largest s in [0, hi] with G[j][s] <= rem   (G[j][.] is non-decreasing, G[j][0] = 0 <= rem)
__device__ __forceinline__ int mcb_search_column(const int* __restrict__ G, int ldg, int j, int hi, int rem, int top_step)
{
    int s = 0;
    for (int step = top_step; step >= 1; step >>= 1) {
        int t = s + step;
        if (t <= hi && mcb_ldG(G, ldg, j, t) <= rem) s = t;
    }
    return s;
}

// Algorithm 2 result via the combinatorial number system: prefix sums S[0..M-1] of the
// configuration with index idx in the space of Np particles (nc_p = N_c(Np, M)).  idx must be in [0, nc_p).
template <int MT>
__device__ __forceinline__ void mcb_unrank_prefix(const int* __restrict__ G, int ldg, int Mrt, int Np, int nc_p,
                                                  int idx, int top_step, int* S)
{
    const int M = MT ? MT : Mrt;
    int rem = nc_p - 1 - idx;
    S[M - 1] = Np;
    int hi = Np;
#pragma unroll
    for (int j = MTraits<MT>::CAP - 2; j >= 1; --j) {
        if (j <= M - 2) {
            int s = mcb_search_column(G, ldg, j, hi, rem, top_step);
            rem -= mcb_ldG(G, ldg, j, s);
            S[j] = s;
            hi = s;
        }
    }
    if (M >= 2) S[0] = rem;            // G[0][s] = s
}

__host__ __device__ inline int mcb_top_step(int N)
{
    int t = 1;
    while (t * 2 <= N) t *= 2;
    return t;
}
