// mcb_maps.cu -- single- and double-jump index maps, written as coalesced int32 planes.
//
// Device layouts (row stride ld = nc rounded up to 64 entries):
//   Map1: plane (k*M + l), entry b  =  index of n^(b) - e_k + e_l, or -1 if n_k = 0          (readings A12, A13)
//   Map2: plane (pair(k<=s)*P + pair(q<=l)), entry b = index of n^(b) - e_k - e_s + e_q + e_l, or -1 if the
//         removal is not allowed                                                              (reading A15)
// One thread per configuration b: threads of a warp write consecutive entries of the same plane.  The occupations come
// from the hashing table when it is attached (2 M bytes read per configuration against 4 M^2 / 4 P^2 written), otherwise
// from Algorithm 2 (column searches): with the table the kernels are HBM-write bound.
#include "mcb_device.cuh"

#define MCB_DISPATCH_M(M, CALL)                                                                          \
    switch (M) {                                                                                         \
    case 1:  { constexpr int MT = 1;  CALL; } break;  case 2:  { constexpr int MT = 2;  CALL; } break;   \
    case 3:  { constexpr int MT = 3;  CALL; } break;  case 4:  { constexpr int MT = 4;  CALL; } break;   \
    case 5:  { constexpr int MT = 5;  CALL; } break;  case 6:  { constexpr int MT = 6;  CALL; } break;   \
    case 7:  { constexpr int MT = 7;  CALL; } break;  case 8:  { constexpr int MT = 8;  CALL; } break;   \
    case 9:  { constexpr int MT = 9;  CALL; } break;  case 10: { constexpr int MT = 10; CALL; } break;   \
    case 11: { constexpr int MT = 11; CALL; } break;  case 12: { constexpr int MT = 12; CALL; } break;   \
    default: { constexpr int MT = 0;  CALL; } break;                                                     \
    }

// A single jump k -> l changes the prefix sums S_j by -1 on [k, l) (k < l) or by +1 on [l, k) (k > l), so
//   index' = b + sum_{j in [k,l)} (G[j][S_j] - G[j][S_j - 1])      (k < l)
//   index' = b - sum_{j in [l,k)} (G[j][S_j + 1] - G[j][S_j])      (k > l)
// i.e. two prefix-sum arrays per configuration and one subtraction per target.
// prefix sums S_j of configuration b: from the hashing table (occ != NULL) or by Algorithm 2
template <int MT>
__device__ __forceinline__ void map_prefix(const McbDev& d, const int M, const int b, const uint16_t* __restrict__ occ, const long long ldo, int* S)
{
    if (occ != nullptr) {
        int run = 0;
#pragma unroll
        for (int j = 0; j < MTraits<MT>::CAP; ++j) if (j < M) { run += (int)__ldg(occ + (long long)j * ldo + b); S[j] = run; }
    } else {
        mcb_unrank_prefix<MT>(d.G, d.ldg, M, d.N, d.nc, b, mcb_top_step(d.N), S);
    }
}

template <int MT>
__global__ void __launch_bounds__(256) k_map1(McbDev d, int* __restrict__ out, long long ld, const uint16_t* __restrict__ occ, long long ldo)
{
    constexpr int CAP = MTraits<MT>::CAP;
    const int M = MT ? MT : d.M;
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= d.nc) return;
    int S[CAP];
    map_prefix<MT>(d, M, b, occ, ldo, S);
    int PM[CAP], PP[CAP];                  // PM[x] = sum_{j<x} dm[j], PP[x] = sum_{j<x} dp[j]
    int pm = 0, pp = 0;
#pragma unroll
    for (int j = 0; j < CAP; ++j) {
        if (j < M) {
            PM[j] = pm; PP[j] = pp;
            if (j <= M - 2) {
                int g0 = mcb_ldG(d.G, d.ldg, j, S[j]);
                int gm = mcb_ldG(d.G, d.ldg, j, S[j] > 0 ? S[j] - 1 : 0);
                int gp = mcb_ldG(d.G, d.ldg, j, S[j] < d.N ? S[j] + 1 : d.N);
                pm += g0 - gm; pp += gp - g0;
            }
        }
    }
#pragma unroll
    for (int k = 0; k < CAP; ++k) {
        if (k < M) {
            const int nk = S[k] - (k ? S[k - 1] : 0);
#pragma unroll
            for (int l = 0; l < CAP; ++l) {
                if (l < M) {
                    int v = -1;
                    if (nk >= 1) v = (k <= l) ? b + (PM[l] - PM[k]) : b - (PP[k] - PP[l]);
                    out[(long long)(k * M + l) * ld + b] = v;
                }
            }
        }
    }
}

// Double jump: with S' the prefix sums of the intermediate m = n - e_k - e_s (S'_j = S_j - [j>=k] - [j>=s]),
// the target m + e_q + e_l (q <= l) has prefix sums S'_j (j < q), S'_j + 1 (q <= j < l), S'_j + 2 (j >= l), so
//   index = nc - 1 - X[q] - Y[l],  X[q] = sum_{j<q} (A0[j] - A1[j]),  Y[l] = sum_{j<l} A1[j] + sum_{j>=l} A2[j],
//   Ai[j] = G[j][S'_j + i].
template <int MT>
__global__ void __launch_bounds__(128) k_map2(McbDev d, int* __restrict__ out, long long ld, const uint16_t* __restrict__ occ, long long ldo)
{
    constexpr int CAP = MTraits<MT>::CAP;
    const int M = MT ? MT : d.M;
    const int P = M * (M + 1) / 2;
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= d.nc) return;
    int S[CAP];
    map_prefix<MT>(d, M, b, occ, ldo, S);
    int a = 0;                                            // removal pair index
    for (int k = 0; k < M; ++k) {
        for (int s = k; s < M; ++s, ++a) {
            int nk = 0, ns = 0;
#pragma unroll
            for (int j = 0; j < CAP; ++j) if (j < M) {
                int nj = S[j] - (j ? S[j - 1] : 0);
                nk = (j == k) ? nj : nk; ns = (j == s) ? nj : ns;
            }
            const bool ok = (k == s) ? (nk >= 2) : (nk >= 1 && ns >= 1);
            int* plane = out + (long long)a * P * ld + b;
            if (!ok) {
                for (int c = 0; c < P; ++c) plane[(long long)c * ld] = -1;
                continue;
            }
            int X[CAP], Y[CAP];
            int A1[CAP], A2[CAP];
            int x = 0;
#pragma unroll
            for (int j = 0; j < CAP; ++j) if (j < M) {
                X[j] = x;
                if (j <= M - 2) {
                    int sp = S[j] - (j >= k) - (j >= s);          // >= 0 because the removal is allowed
                    int a0 = mcb_ldG(d.G, d.ldg, j, sp);
                    A1[j] = mcb_ldG(d.G, d.ldg, j, sp + 1);
                    A2[j] = mcb_ldG(d.G, d.ldg, j, sp + 2);
                    x += a0 - A1[j];
                } else { A1[j] = 0; A2[j] = 0; }
            }
            int suf = 0;                                  // sum_{j>=l} A2[j]
            int tot1 = 0;
#pragma unroll
            for (int j = 0; j < CAP; ++j) if (j < M) tot1 += A1[j];
            int pre = tot1;                               // sum_{j<l} A1[j], filled from l = M-1 down
#pragma unroll
            for (int l = CAP - 1; l >= 0; --l) if (l < M) {
                pre -= A1[l];                             // now sum_{j<l} A1[j]  (A1[M-1] = 0)
                suf += A2[l];                             // now sum_{j>=l} A2[j] (A2[M-1] = 0)
                Y[l] = pre + suf;
            }
            int c = 0;
#pragma unroll
            for (int q = 0; q < CAP; ++q) if (q < M) {
#pragma unroll
                for (int l = 0; l < CAP; ++l) if (l < M && l >= q) {
                    plane[(long long)c * ld] = d.nc - 1 - X[q] - Y[l];
                    ++c;
                }
            }
        }
    }
}

int mcb_launch_map1(const mcb_space* sp, int* d_out, long long ld, cudaStream_t st)
{
    const int threads = 256;
    const unsigned blocks = (unsigned)((sp->nc + threads - 1) / threads);
    MCB_DISPATCH_M(sp->M, (k_map1<MT><<<blocks, threads, 0, st>>>(sp->dev, d_out, ld, sp->d_fock ? sp->fock.occ : nullptr, sp->fock.ld)));
    MCB_CHECK_LAUNCH();
    return MCB_OK;
}

int mcb_launch_map2(const mcb_space* sp, int* d_out, long long ld, cudaStream_t st)
{
    const int threads = 128;
    const unsigned blocks = (unsigned)((sp->nc + threads - 1) / threads);
    MCB_DISPATCH_M(sp->M, (k_map2<MT><<<blocks, threads, 0, st>>>(sp->dev, d_out, ld, sp->d_fock ? sp->fock.occ : nullptr, sp->fock.ld)));
    MCB_CHECK_LAUNCH();
    return MCB_OK;
}
