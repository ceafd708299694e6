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

// ---- Algorithms 1 and 2, batched: one thread per index / configuration --------------------------------------
// The ABI layout is row-major int32 [batch][M].  Rows are staged through shared memory (row stride M | 1: odd, so the
// per-thread row accesses are bank-conflict free) and move to / from global memory as 16-byte vectors of the contiguous
// 256 x M block, so that both sides of the kernel are streaming accesses.
__device__ __forceinline__ int hash_rows_here(long long batch, long long base, int threads)
{
    long long r = batch - base;
    return (int)(r > threads ? threads : r);
}

// Algorithm 2: a thread takes UR_SPAN consecutive entries of the batch.  The first is unranked by the column searches; an entry
// that is the successor of the one before it (idx[i] = idx[i-1] + 1: every entry of an identity-range batch, the common way
// to list a whole space) is stepped to with the successor rule of the order of Eq. (14) instead (see k_fock_table8) -- one
// search per UR_SPAN entries; anything else is searched on its own.  Same results either way.
#define UR_SPAN 4
template <int MT>
__global__ void __launch_bounds__(256) k_unrank(McbDev d, const int* __restrict__ idx, long long batch, int* __restrict__ occ, int vec_ok, int idx_vec_ok)
{
    const int M = MT ? MT : d.M;
    const int MP = M | 1;
    constexpr int CAP = MTraits<MT>::CAP;
    extern __shared__ int s_rows[];                       // [blockDim.x * UR_SPAN][MP]
    const long long base = (long long)blockIdx.x * blockDim.x * UR_SPAN;
    const long long i0 = base + (long long)threadIdx.x * UR_SPAN;
    const int top = mcb_top_step(d.N);
    if (i0 < batch) {
        int bb[UR_SPAN];
        if (idx_vec_ok && i0 + UR_SPAN <= batch) {
            const int4 q = __ldcs(reinterpret_cast<const int4*>(idx + i0));
            bb[0] = q.x; bb[1] = q.y; bb[2] = q.z; bb[3] = q.w;
        } else {
#pragma unroll
            for (int e = 0; e < UR_SPAN; ++e) bb[e] = i0 + e < batch ? idx[i0 + e] : -1;
        }
        int n[CAP];
        bool have = false;                                // n holds the configuration of the previous entry
#pragma unroll
        for (int e = 0; e < UR_SPAN; ++e) {
            if (i0 + e >= batch) break;
            const int b = bb[e];
            int* row = s_rows + (threadIdx.x * UR_SPAN + e) * MP;
            if (b < 0 || b >= d.nc) {
#pragma unroll
                for (int j = 0; j < CAP; ++j) if (j < M) row[j] = -1;
                have = false;
                continue;
            }
            if (have && b == bb[e > 0 ? e - 1 : 0] + 1) {
                if (M >= 2 && n[0] >= 1) { n[0] -= 1; n[1] += 1; }          // inside a run: the common case
                else {
                    int S = n[0], jstar = 0;
#pragma unroll
                    for (int j = 1; j < CAP; ++j) if (j < M) { if (jstar == 0 && S >= 1) jstar = j; if (jstar == 0) S += n[j]; }
#pragma unroll
                    for (int j = 1; j < CAP; ++j) if (j < M) { if (j < jstar) n[j] = 0; else if (j == jstar) n[j] += 1; }
                    n[0] = S - 1;
                }
            } else {
                int S[CAP];
                mcb_unrank_prefix<MT>(d.G, d.ldg, M, d.N, d.nc, b, top, S);
                int prev = 0;
#pragma unroll
                for (int j = 0; j < CAP; ++j) if (j < M) { n[j] = S[j] - prev; prev = S[j]; }
                have = true;
            }
#pragma unroll
            for (int j = 0; j < CAP; ++j) if (j < M) row[j] = n[j];
        }
    }
    __syncthreads();
    const int total = hash_rows_here(batch, base, blockDim.x * UR_SPAN) * M;
    int* out = occ + base * M;
    const int nvec = vec_ok ? total >> 2 : 0;
    for (int v = threadIdx.x; v < nvec; v += blockDim.x) {
        int x[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) { const int e = 4 * v + k; x[k] = s_rows[(e / M) * MP + (e % M)]; }
        reinterpret_cast<int4*>(out)[v] = make_int4(x[0], x[1], x[2], x[3]);
    }
    for (int e = 4 * nvec + threadIdx.x; e < total; e += blockDim.x) out[e] = s_rows[(e / M) * MP + (e % M)];
}

template <int MT>
__global__ void __launch_bounds__(256) k_rank(McbDev d, const int* __restrict__ occ, long long batch, int* __restrict__ idx, int vec_ok)
{
    const int M = MT ? MT : d.M;
    const int MP = M | 1;
    extern __shared__ int s_rows[];
    const long long base = (long long)blockIdx.x * blockDim.x;
    if (MT != 0 && MT % 4 == 0 && vec_ok) {
        // a row is MT / 4 whole 16-byte vectors: every thread loads its own row (a warp still reads one contiguous block)
        const long long i = base + threadIdx.x;
        if (i >= batch) return;
        const int4* rowv = reinterpret_cast<const int4*>(occ + i * M);
        int S = 0, acc = 0;
        bool ok = true;
#pragma unroll
        for (int v = 0; v < (MT ? MT : 4) / 4; ++v) {
            const int4 q = __ldcs(rowv + v);
            const int x[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int j = 4 * v + k;
                ok = ok && x[k] >= 0 && x[k] <= d.N - S;
                S += ok ? x[k] : 0;
                if (j <= M - 2) acc += mcb_ldG(d.G, d.ldg, j, S);
            }
        }
        ok = ok && S == d.N;
        idx[i] = ok ? d.nc - 1 - acc : -1;
        return;
    }
    const int total = hash_rows_here(batch, base, blockDim.x) * M;
    const int* in = occ + base * M;
    const int nvec = vec_ok ? total >> 2 : 0;
    for (int v = threadIdx.x; v < nvec; v += blockDim.x) {
        const int4 q = __ldcs(reinterpret_cast<const int4*>(in) + v);
        const int x[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) { const int e = 4 * v + k; s_rows[(e / M) * MP + (e % M)] = x[k]; }
    }
    for (int e = 4 * nvec + threadIdx.x; e < total; e += blockDim.x) s_rows[(e / M) * MP + (e % M)] = in[e];
    __syncthreads();
    const long long i = base + threadIdx.x;
    if (i >= batch) return;
    const int* row = s_rows + threadIdx.x * MP;
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

// Same table for compile-time M: a thread unranks the first of FT_SPAN consecutive indices (binary search of the columns
// of G) and STEPS through the rest with the successor rule of the order of Eq. (14) (n_1 is the least significant digit,
// n_0 the remainder): with j* the smallest j >= 1 such that S_{j*-1} >= 1,
//     n_{j*} += 1,   n_1 .. n_{j*-1} = 0,   n_0 = S_{j*-1} - 1.
// The FT_W occupations of an orbital leave as one 16-byte store: HBM-write bound instead of search bound.  (Measured: 16 or 32
// configurations per thread are slower -- the stores of a warp are then strided and at M = 12 the packing registers halve
// the occupancy: 1.26 TB/s against 2.2 TB/s at configs[4].)
#define FT_W 8                         // configurations per store group (16 bytes per orbital: a warp writes 512 contiguous bytes)
#define FT_GROUPS 1                    // store groups per thread: one column search per FT_SPAN configurations
#define FT_SPAN (FT_W * FT_GROUPS)
template <int MT>
__global__ void __launch_bounds__(256) k_fock_table8(McbDev d, int Np, int nc_p, uint16_t* __restrict__ out, long long ld)
{
    static_assert(MT >= 1, "compile-time M");
    constexpr int M = MT;
    const long long bfirst_ll = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * FT_SPAN;
    if (bfirst_ll >= nc_p) return;
    const int bfirst = (int)bfirst_ll;
    int n[M];
    {
        int S[M];
        mcb_unrank_prefix<MT>(d.G, d.ldg, M, Np, nc_p, bfirst, mcb_top_step(Np > 0 ? Np : 1), S);
        int prev = 0;
#pragma unroll
        for (int j = 0; j < M; ++j) { n[j] = S[j] - prev; prev = S[j]; }
    }
#pragma unroll 1
    for (int grp = 0; grp < FT_GROUPS; ++grp) {
        const int b0 = bfirst + FT_W * grp;
        if (b0 >= nc_p) return;
        unsigned pk[M][FT_W / 2];
#pragma unroll
        for (int j = 0; j < M; ++j)
#pragma unroll
            for (int w = 0; w < FT_W / 2; ++w) pk[j][w] = 0u;
        const int cnt = min(FT_W, nc_p - b0);
#pragma unroll
        for (int i = 0; i < FT_W; ++i) {
            if (i < cnt) {
#pragma unroll
                for (int j = 0; j < M; ++j) pk[j][i >> 1] |= (unsigned)n[j] << (16 * (i & 1));
            }
            if (b0 + i + 1 < nc_p) {                         // successor (the last one of a group feeds the next group)
                if (M >= 2 && n[0] >= 1) { n[0] -= 1; n[1] += 1; }          // inside a run: the common case
                else {
                    int S = n[0], jstar = 0;
#pragma unroll
                    for (int j = 1; j < M; ++j) { if (jstar == 0 && S >= 1) jstar = j; if (jstar == 0) S += n[j]; }
#pragma unroll
                    for (int j = 1; j < M; ++j) { if (j < jstar) n[j] = 0; else if (j == jstar) n[j] += 1; }
                    n[0] = S - 1;
                }
            }
        }
        if (cnt == FT_W) {
#pragma unroll
            for (int j = 0; j < M; ++j) {
                uint4* dst = reinterpret_cast<uint4*>(out + (long long)j * ld + b0);
#pragma unroll
                for (int w = 0; w < FT_W / 8; ++w) dst[w] = make_uint4(pk[j][4 * w], pk[j][4 * w + 1], pk[j][4 * w + 2], pk[j][4 * w + 3]);
            }
        } else {
#pragma unroll
            for (int j = 0; j < M; ++j)
#pragma unroll
                for (int i = 0; i < FT_W; ++i)
                    if (i < cnt) out[(long long)j * ld + b0 + i] = (uint16_t)((pk[j][i >> 1] >> (16 * (i & 1))) & 0xffffu);
        }
    }
}

int mcb_launch_unrank(const mcb_space* sp, const int* d_idx, long long batch, int* d_occ, cudaStream_t st)
{
    const int threads = sp->M <= 12 ? 256 : 64;                          // (rows of a block in shared memory: 4 x threads x (M | 1) ints)
    const long long per_block = (long long)threads * UR_SPAN;
    const long long blocks = (batch + per_block - 1) / per_block;
    if (blocks > 2147483647LL) return MCB_ERANGE;
    const size_t smem = (size_t)per_block * (sp->M | 1) * sizeof(int);
    const int vec_ok = ((uintptr_t)d_occ % 16) == 0, idx_vec_ok = ((uintptr_t)d_idx % 16) == 0;
    if (smem > 48 * 1024) {
        MCB_DISPATCH_M(sp->M, (cudaFuncSetAttribute(k_unrank<MT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)));
    }
    MCB_DISPATCH_M(sp->M, (k_unrank<MT><<<(unsigned)blocks, threads, smem, st>>>(sp->dev, d_idx, batch, d_occ, vec_ok, idx_vec_ok)));
    MCB_CHECK_LAUNCH();
    return MCB_OK;
}

int mcb_launch_rank(const mcb_space* sp, const int* d_occ, long long batch, int* d_idx, cudaStream_t st)
{
    const int threads = 256;
    const long long blocks = (batch + threads - 1) / threads;
    if (blocks > 2147483647LL) return MCB_ERANGE;
    const size_t smem = (size_t)threads * (sp->M | 1) * sizeof(int);
    const int vec_ok = ((uintptr_t)d_occ % 16) == 0;
    MCB_DISPATCH_M(sp->M, (k_rank<MT><<<(unsigned)blocks, threads, smem, st>>>(sp->dev, d_occ, batch, d_idx, vec_ok)));
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
        const unsigned blocks = (unsigned)(((n + FT_SPAN - 1) / FT_SPAN + threads - 1) / threads);
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
