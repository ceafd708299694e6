// mcb_hash.cu -- batched Algorithm 1 / Algorithm 2 and the hashing table.
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

// ---- Algorithm 2, batched: one thread per index ---------------------------------------------------------
// Output row-major int32 [batch][M] (ABI layout).  Rows are staged through shared memory so that the global
// stores of a warp are contiguous (32 rows x M ints) instead of M-strided.
template <int MT>
__global__ void __launch_bounds__(256) k_unrank(McbDev d, const int* __restrict__ idx, long long batch, int* __restrict__ occ)
{
    const int M = MT ? MT : d.M;
    extern __shared__ int s_rows[];                       // [blockDim.x][M]
    const long long base = (long long)blockIdx.x * blockDim.x;
    const long long i = base + threadIdx.x;
    const int top = mcb_top_step(d.N);
    if (i < batch) {
        int b = idx[i];
        int S[MTraits<MT>::CAP];
        int* row = s_rows + threadIdx.x * M;
        if (b < 0 || b >= d.nc) {
#pragma unroll
            for (int j = 0; j < MTraits<MT>::CAP; ++j) if (j < M) row[j] = -1;
        } else {
            mcb_unrank_prefix<MT>(d.G, d.ldg, M, d.N, d.nc, b, top, S);
            int prev = 0;
#pragma unroll
            for (int j = 0; j < MTraits<MT>::CAP; ++j) if (j < M) { row[j] = S[j] - prev; prev = S[j]; }
        }
    }
    __syncthreads();
    long long rows_here = batch - base;
    if (rows_here > blockDim.x) rows_here = blockDim.x;
    const int total = (int)rows_here * M;
    int* out = occ + base * M;
    for (int t = threadIdx.x; t < total; t += blockDim.x) out[t] = s_rows[t];
}

// ---- Algorithm 1, batched: one thread per configuration ---------------------------------------------------
template <int MT>
__global__ void __launch_bounds__(256) k_rank(McbDev d, const int* __restrict__ occ, long long batch, int* __restrict__ idx)
{
    const int M = MT ? MT : d.M;
    extern __shared__ int s_rows[];
    const long long base = (long long)blockIdx.x * blockDim.x;
    long long rows_here = batch - base;
    if (rows_here > blockDim.x) rows_here = blockDim.x;
    const int total = (int)rows_here * M;
    const int* in = occ + base * M;
    for (int t = threadIdx.x; t < total; t += blockDim.x) s_rows[t] = in[t];
    __syncthreads();
    const long long i = base + threadIdx.x;
    if (i >= batch) return;
    const int* row = s_rows + threadIdx.x * M;
    int S = 0, acc = 0;
    bool ok = true;
#pragma unroll
    for (int j = 0; j < MTraits<MT>::CAP; ++j) {
        if (j < M) {
            int nj = row[j];
            ok = ok && nj >= 0 && nj <= d.N - S;            // also guards the table look-up range
            S += ok ? nj : 0;
            if (j <= M - 2) acc += mcb_ldG(d.G, d.ldg, j, S);
        }
    }
    ok = ok && S == d.N;
    idx[i] = ok ? d.nc - 1 - acc : -1;
}

// ---- hashing table: all occupation vectors of the (N - removed)-particle space, uint16 SoA [j][b] ---------
template <int MT>
__global__ void __launch_bounds__(256) k_fock_table(McbDev d, int Np, int nc_p, uint16_t* __restrict__ out, long long ld)
{
    const int M = MT ? MT : d.M;
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nc_p) return;
    int S[MTraits<MT>::CAP];
    mcb_unrank_prefix<MT>(d.G, d.ldg, M, Np, nc_p, b, mcb_top_step(Np > 0 ? Np : 1), S);
    int prev = 0;
#pragma unroll
    for (int j = 0; j < MTraits<MT>::CAP; ++j)
        if (j < M) { out[(long long)j * ld + b] = (uint16_t)(S[j] - prev); prev = S[j]; }
}

// Same table for compile-time M: a thread unranks the first of 8 consecutive indices (binary search of the columns
// of G) and STEPS to the next seven with the successor rule of the order of Eq. (14) (n_1 is the least significant
// digit, n_0 the remainder): with j* the smallest j >= 1 such that S_{j*-1} >= 1,
//     n_{j*} += 1,   n_1 .. n_{j*-1} = 0,   n_0 = S_{j*-1} - 1.
// The 8 occupations of an orbital leave as one 16-byte store: HBM-write bound instead of search bound.
template <int MT>
__global__ void __launch_bounds__(256) k_fock_table8(McbDev d, int Np, int nc_p, uint16_t* __restrict__ out, long long ld)
{
    static_assert(MT >= 1, "compile-time M");
    constexpr int M = MT;
    const int b0 = (blockIdx.x * blockDim.x + threadIdx.x) * 8;
    if (b0 >= nc_p) return;
    int n[M];
    {
        int S[M];
        mcb_unrank_prefix<MT>(d.G, d.ldg, M, Np, nc_p, b0, mcb_top_step(Np > 0 ? Np : 1), S);
        int prev = 0;
#pragma unroll
        for (int j = 0; j < M; ++j) { n[j] = S[j] - prev; prev = S[j]; }
    }
    unsigned pk[M][4];
#pragma unroll
    for (int j = 0; j < M; ++j) { pk[j][0] = pk[j][1] = pk[j][2] = pk[j][3] = 0u; }
    const int cnt = min(8, nc_p - b0);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        if (i < cnt) {
#pragma unroll
            for (int j = 0; j < M; ++j) pk[j][i >> 1] |= (unsigned)n[j] << (16 * (i & 1));
        }
        if (i + 1 < cnt) {                                   // successor
            int S = n[0], jstar = 0;
#pragma unroll
            for (int j = 1; j < M; ++j) { if (jstar == 0 && S >= 1) jstar = j; if (jstar == 0) S += n[j]; }
#pragma unroll
            for (int j = 1; j < M; ++j) { if (j < jstar) n[j] = 0; else if (j == jstar) n[j] += 1; }
            n[0] = S - 1;
        }
    }
    if (cnt == 8) {
#pragma unroll
        for (int j = 0; j < M; ++j)
            *reinterpret_cast<uint4*>(out + (long long)j * ld + b0) = make_uint4(pk[j][0], pk[j][1], pk[j][2], pk[j][3]);
    } else {
#pragma unroll
        for (int j = 0; j < M; ++j)
#pragma unroll
            for (int i = 0; i < 8; ++i)
                if (i < cnt) out[(long long)j * ld + b0 + i] = (uint16_t)((pk[j][i >> 1] >> (16 * (i & 1))) & 0xffffu);
    }
}

int mcb_launch_unrank(const mcb_space* sp, const int* d_idx, long long batch, int* d_occ, cudaStream_t st)
{
    const int threads = 256;
    const long long blocks = (batch + threads - 1) / threads;
    if (blocks > 2147483647LL) return MCB_ERANGE;
    const size_t smem = (size_t)threads * sp->M * sizeof(int);
    MCB_DISPATCH_M(sp->M, (k_unrank<MT><<<(unsigned)blocks, threads, smem, st>>>(sp->dev, d_idx, batch, d_occ)));
    MCB_CHECK_LAUNCH();
    return MCB_OK;
}

int mcb_launch_rank(const mcb_space* sp, const int* d_occ, long long batch, int* d_idx, cudaStream_t st)
{
    const int threads = 256;
    const long long blocks = (batch + threads - 1) / threads;
    if (blocks > 2147483647LL) return MCB_ERANGE;
    const size_t smem = (size_t)threads * sp->M * sizeof(int);
    MCB_DISPATCH_M(sp->M, (k_rank<MT><<<(unsigned)blocks, threads, smem, st>>>(sp->dev, d_occ, batch, d_idx)));
    MCB_CHECK_LAUNCH();
    return MCB_OK;
}

int mcb_launch_fock_table(const mcb_space* sp, int removed, uint16_t* d_out, long long ld, cudaStream_t st)
{
    const int Np = sp->N - removed;
    const long long n = removed == 0 ? sp->nc : sp->nc2;
    if (Np < 0 || n <= 0) return MCB_OK;
    const int threads = 256;
    if (sp->M <= 12 && (ld % 8) == 0 && ((uintptr_t)d_out % 16) == 0) {
        const unsigned blocks = (unsigned)(((n + 7) / 8 + threads - 1) / threads);
        switch (sp->M) {
#define MCB_FT8(MM) case MM: k_fock_table8<MM><<<blocks, threads, 0, st>>>(sp->dev, Np, (int)n, d_out, ld); break;
        MCB_FT8(1) MCB_FT8(2) MCB_FT8(3) MCB_FT8(4) MCB_FT8(5) MCB_FT8(6) MCB_FT8(7) MCB_FT8(8) MCB_FT8(9) MCB_FT8(10) MCB_FT8(11) MCB_FT8(12)
#undef MCB_FT8
        }
    } else {
        const unsigned blocks = (unsigned)((n + threads - 1) / threads);
        MCB_DISPATCH_M(sp->M, (k_fock_table<MT><<<blocks, threads, 0, st>>>(sp->dev, Np, (int)n, d_out, ld)));
    }
    MCB_CHECK_LAUNCH();
    return MCB_OK;
}
