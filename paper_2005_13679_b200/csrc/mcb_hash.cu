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
    const unsigned blocks = (unsigned)((n + threads - 1) / threads);
    MCB_DISPATCH_M(sp->M, (k_fock_table<MT><<<blocks, threads, 0, st>>>(sp->dev, Np, (int)n, d_out, ld)));
    MCB_CHECK_LAUNCH();
    return MCB_OK;
}
