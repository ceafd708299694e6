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

// log2((j+1)!), j = 0..31
__device__ __constant__ float c_mcb_log2fact[32] = {
    0.0000000f, 1.0000000f, 2.5849625f, 4.5849625f, 6.9068906f, 9.4918531f, 12.2992080f, 15.2992080f, 18.4691330f, 21.7910611f,
    25.2504927f, 28.8354552f, 32.5358950f, 36.3432499f, 40.2501405f, 44.2501405f, 48.3376033f, 52.5075283f, 56.7554558f,
    61.0773839f, 65.4697013f, 69.9291330f, 74.4526949f, 79.0376574f, 83.6815136f, 88.3819533f, 93.1368408f, 97.9441958f,
    102.8021767f, 107.7090673f, 112.6632637f, 117.6632637f};

// largest s in [0, hi] with G[j][s] <= rem   (G[j][.] is non-decreasing, G[j][0] = 0 <= rem).
// Short columns: binary search (log2 hi dependent probes).  Long columns (many particles): the probes of a warp scatter over
// the whole column and the kernel becomes bound by L1 wavefronts, so the search starts from the inverse of
// G[j][s] = s (s+1) .. (s+j) / (j+1)! ~ (s + j/2)^(j+1) / (j+1)!  evaluated in fp32 and is corrected by walking: whatever the
// guess, the two loops end at the exact answer (usually after two or three probes).
__device__ __forceinline__ int mcb_search_column(const int* __restrict__ G, int ldg, int j, int hi, int rem, int top_step)
{
    if (top_step <= 16) {
        int s = 0;
        for (int step = top_step; step >= 1; step >>= 1) {
            int t = s + step;
            if (t <= hi && mcb_ldG(G, ldg, j, t) <= rem) s = t;
        }
        return s;
    }
    if (rem == 0 || hi == 0) return 0;
    const float x = exp2f((__log2f((float)rem) + c_mcb_log2fact[j]) / (float)(j + 1)) - 0.5f * (float)j;
    int s = min(max((int)x, 0), hi);
    while (s > 0 && mcb_ldG(G, ldg, j, s) > rem) --s;
    while (s < hi && mcb_ldG(G, ldg, j, s + 1) <= rem) ++s;
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
