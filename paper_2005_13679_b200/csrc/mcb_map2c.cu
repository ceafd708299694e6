// mcb_map2c.cu -- the paper's COMPACT double-jump map (Fig. 3) and the hc_apply kernel that streams it.
//
// Layout (MCB_MAP2C), as Sec. IV describes it: a table "like a hashing table, though each line has a variable number of
// elements"; line g (configuration index) holds, for every ALLOWED simultaneous removal from orbitals k <= s -- in the
// order k = 0 .. M-1, s = k .. M-1 -- one STRIDE with the indices of the configurations reached by putting the two particles
// back; to find the stride of a given (i, j) one skips "the number of possible simultaneous removals from k and s for every
// k = 0..i and s = k..j-1" strides (Fig. 3: the last removal of its example is 3 strides in).
// A stride here holds the P = M(M+1)/2 UNORDERED replacements (q <= l), in pair order; the paper's M^2 stride stores each
// q != l target twice (reading A15b).  Forbidden removals take no memory: sum_g #allowed(g) = P nc2 strides, i.e.
// 4 P^2 nc2 bytes (configs[3]: 57 GB instead of the 121 GB of the dense MCB_MAP2; configs[4]: 61 GB instead of 188 GB).
//   buffer = [ soff : nc + 1 int64, stride offset of every line (exclusive prefix sum of the allowed-removal counts) ]
//            [ block sums of the scan ][ entries : P nc2 strides x P int32 ]
// Build: k_m2c_count (allowed removals per configuration, per-block sums) -> k_m2c_scan (one block scans the block sums)
//        -> k_m2c_offsets (per-block scan + base) -> k_m2c_fill (one thread per configuration writes its line).
// Apply (MCB_MAPS with this map attached; T folded into Vp, so the table serves alone):
//   P <= 15 (M <= 5)  k_hc_maps2c<M>: one thread per OUTPUT configuration, removal pairs walked in lockstep, the next stride of
//                     the line prefetched into registers before the gathers of the current one (configs[2]: 2.6 ms against
//                     8.0 ms for the lane-group kernel, 2.3 ms for the dense planes);
//   P  > 15           k_hc_maps2c_group<M, 32>: a warp per output configuration walks its line stride by stride, one gather per
//                     lane and stride, partial sums added by shuffles.
// No atomics anywhere.  This is the paper's own fast variant: it streams 4 P^2 nc2 bytes of map per apply.
#include <stdlib.h>
#include <string.h>
#include "mcb_device.cuh"

#define M2C_BLOCK 1024                // configurations per scan block
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

// number of allowed removal pairs of a configuration: (k < s both occupied) + (k == s with n_k >= 2)
__device__ __forceinline__ int m2c_count(const uint16_t* __restrict__ occ, long long ldo, int M, int g)
{
    int nocc = 0, ntwo = 0;
    for (int j = 0; j < M; ++j) {
        const int nj = (int)__ldg(occ + (long long)j * ldo + g);
        nocc += nj >= 1; ntwo += nj >= 2;
    }
    return nocc * (nocc - 1) / 2 + ntwo;
}

__global__ void __launch_bounds__(256) k_m2c_count(McbDev d, const uint16_t* __restrict__ occ, long long ldo, long long* __restrict__ bsum)
{
    __shared__ int s[256];
    const int g0 = blockIdx.x * M2C_BLOCK;
    int acc = 0;
    for (int g = g0 + threadIdx.x; g < min(g0 + M2C_BLOCK, d.nc); g += 256) acc += m2c_count(occ, ldo, d.M, g);
    s[threadIdx.x] = acc;
    __syncthreads();
    for (int o = 128; o >= 1; o >>= 1) { if (threadIdx.x < o) s[threadIdx.x] += s[threadIdx.x + o]; __syncthreads(); }
    if (threadIdx.x == 0) bsum[blockIdx.x] = s[0];
}

// exclusive scan of the block sums, in place, by one block (fixed order)
__global__ void __launch_bounds__(1024) k_m2c_scan(long long* __restrict__ bsum, int nblocks, long long* __restrict__ total)
{
    __shared__ long long s[1024];
    __shared__ long long carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int b0 = 0; b0 < nblocks; b0 += 1024) {
        const int i = b0 + threadIdx.x;
        const long long v = i < nblocks ? bsum[i] : 0;
        s[threadIdx.x] = v;
        __syncthreads();
        for (int o = 1; o < 1024; o <<= 1) {
            const long long t = threadIdx.x >= o ? s[threadIdx.x - o] : 0;
            __syncthreads();
            s[threadIdx.x] += t;
            __syncthreads();
        }
        if (i < nblocks) bsum[i] = carry + s[threadIdx.x] - v;          // exclusive
        __syncthreads();
        if (threadIdx.x == 1023) carry += s[1023];
        __syncthreads();
    }
    if (threadIdx.x == 0) *total = carry;
}

// soff[g] = base of the block + exclusive scan inside the block; soff[nc] = total
__global__ void __launch_bounds__(256) k_m2c_offsets(McbDev d, const uint16_t* __restrict__ occ, long long ldo, const long long* __restrict__ bsum,
                                                    const long long* __restrict__ total, long long* __restrict__ soff)
{
    __shared__ int s[256];
    __shared__ int carry;
    const int g0 = blockIdx.x * M2C_BLOCK;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int r = 0; r < M2C_BLOCK / 256; ++r) {
        const int g = g0 + r * 256 + threadIdx.x;
        const int v = g < d.nc ? m2c_count(occ, ldo, d.M, g) : 0;
        s[threadIdx.x] = v;
        __syncthreads();
        for (int o = 1; o < 256; o <<= 1) {
            const int t = threadIdx.x >= o ? s[threadIdx.x - o] : 0;
            __syncthreads();
            s[threadIdx.x] += t;
            __syncthreads();
        }
        if (g < d.nc) soff[g] = bsum[blockIdx.x] + carry + s[threadIdx.x] - v;
        __syncthreads();
        if (threadIdx.x == 255) carry += s[255];
        __syncthreads();
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) soff[d.nc] = *total;
}

// ---- fill: one thread per configuration writes its line, stride after stride (the index arithmetic of k_map2, mcb_maps.cu) ----
// A stride is P consecutive int32 (8-byte aligned when P is even: stored as int2).  The lines of neighbouring threads follow
// each other in memory, so every sector is completed by the warp within a few strides and leaves L2 once.
template <int MT>
__global__ void __launch_bounds__(128) k_m2c_fill(McbDev d, const uint16_t* __restrict__ occ, long long ldo, const long long* __restrict__ soff,
                                                 int* __restrict__ entries)
{
    constexpr int CAP = MTraits<MT>::CAP;
    const int M = MT ? MT : d.M;
    const int P = M * (M + 1) / 2;
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= d.nc) return;
    int n[CAP], S[CAP];
    {
        int run = 0;
#pragma unroll
        for (int j = 0; j < CAP; ++j) if (j < M) { n[j] = (int)__ldg(occ + (long long)j * ldo + g); run += n[j]; S[j] = run; }
    }
    int* line = entries + soff[g] * P;
    for (int k = 0; k < M; ++k) {
        for (int s = k; s < M; ++s) {
            int nk = 0, ns = 0;
#pragma unroll
            for (int j = 0; j < CAP; ++j) if (j < M) { nk = (j == k) ? n[j] : nk; ns = (j == s) ? n[j] : ns; }
            if ((k == s) ? (nk < 2) : (nk < 1 || ns < 1)) continue;
            int X[CAP], Y[CAP], A1[CAP], A2[CAP];
            int x = 0, tot1 = 0;
#pragma unroll
            for (int j = 0; j < CAP; ++j) if (j < M) {
                X[j] = x;
                if (j <= M - 2) {
                    const int sp = S[j] - (j >= k) - (j >= s);
                    const int a0 = mcb_ldG(d.G, d.ldg, j, sp);
                    A1[j] = mcb_ldG(d.G, d.ldg, j, sp + 1);
                    A2[j] = mcb_ldG(d.G, d.ldg, j, sp + 2);
                    x += a0 - A1[j]; tot1 += A1[j];
                } else { A1[j] = 0; A2[j] = 0; }
            }
            int pre = tot1, suf = 0;
#pragma unroll
            for (int l = CAP - 1; l >= 0; --l) if (l < M) { pre -= A1[l]; suf += A2[l]; Y[l] = pre + suf; }
            if (MT != 0 && (MT * (MT + 1) / 2) % 2 == 0) {
                int2* l2 = reinterpret_cast<int2*>(line);
                int c = 0, first = 0;
#pragma unroll
                for (int q = 0; q < CAP; ++q) if (q < M) {
#pragma unroll
                    for (int l = 0; l < CAP; ++l) if (l < M && l >= q) {
                        const int t = (int)MCB_CHK(d, d.nc - 1 - X[q] - Y[l], d.nc, 602);
                        if (c & 1) __stcs(l2 + (c >> 1), make_int2(first, t)); else first = t;
                        ++c;
                    }
                }
            } else {
                int c = 0;
#pragma unroll
                for (int q = 0; q < CAP; ++q) if (q < M) {
#pragma unroll
                    for (int l = 0; l < CAP; ++l) if (l < M && l >= q) { __stcs(line + c, (int)MCB_CHK(d, d.nc - 1 - X[q] - Y[l], d.nc, 602)); ++c; }
                }
            }
            line += P;
        }
    }
}

// ---- apply ------------------------------------------------------------------------------------------------------------
struct M2cArgs {
    McbDev d;
    McbFockView fock;
    const double2* C;
    double2* HC;
    const double2* Vp;         // [P][P], T folded in (device)
    const long long* soff;
    const int* entries;
    long long nstrides;        // P nc2 strides in the table
};

// One thread per output configuration g.  The removal pairs (k <= s) are walked in lockstep by the whole block (uniform
// coefficient row Vp[a][.] from shared memory, broadcast); a thread whose configuration allows the pair consumes the next
// stride of its line.  The line is contiguous, so the stride AFTER the current one is loaded before the current one's gathers
// are issued: no gather waits for the map load in front of it.  Lines of neighbouring threads follow each other in memory:
// every sector of the table is fetched once from DRAM (L2 holds the few strides a warp is working on).
#define M2C_THREADS 128
template <int M>
__global__ void __launch_bounds__(M2C_THREADS) k_hc_maps2c(const M2cArgs p)
{
    constexpr int P = M * (M + 1) / 2;
    constexpr bool WIDE = P % 2 == 0;                                    // strides are 8-byte aligned: int2 loads
    constexpr bool PREFETCH = P <= 15;                                   // two target buffers in registers
    extern __shared__ double2 m2c_smem[];
    double2* sV = m2c_smem;                                              // [P*P]
    const McbDev& d = p.d;
    for (int i = threadIdx.x; i < P * P; i += M2C_THREADS) sV[i] = p.Vp[i];
    __syncthreads();
    const int g = blockIdx.x * M2C_THREADS + threadIdx.x;
    if (g >= d.nc) return;
    int n[M];
#pragma unroll
    for (int j = 0; j < M; ++j) n[j] = (int)__ldg(p.fock.occ + (long long)j * p.fock.ld + g);
    const int* line = p.entries + p.soff[g] * (long long)P;
    const int* const last = p.entries + (p.nstrides - 1) * (long long)P;   // the last stride of the table (prefetch clamp)
    auto load_stride = [&](int (&t)[P], const int* src) {
        if (WIDE) {
#pragma unroll
            for (int c = 0; c < P; c += 2) { const int2 v = __ldg(reinterpret_cast<const int2*>(src) + (c >> 1)); t[c] = v.x; t[c + (WIDE ? 1 : 0)] = v.y; }
        } else {
#pragma unroll
            for (int c = 0; c < P; ++c) t[c] = __ldg(src + c);
        }
    };
    int tcur[P], tnext[PREFETCH ? P : 1];
    if (PREFETCH) load_stride(tcur, line < last ? line : last);
    double re = 0.0, im = 0.0;
#pragma unroll 1
    for (int k = 0; k < M; ++k) {
#pragma unroll 1
        for (int s = k; s < M; ++s) {
            int nk = 0, ns = 0;
#pragma unroll
            for (int j = 0; j < M; ++j) { nk = (j == k) ? n[j] : nk; ns = (j == s) ? n[j] : ns; }
            const bool ok = (k == s) ? (nk >= 2) : (nk >= 1 && ns >= 1);
            if (!ok) continue;
            if (PREFETCH) { const int* nx = line + P; load_stride(reinterpret_cast<int (&)[P]>(tnext), nx < last ? nx : last); }
            else load_stride(tcur, line);
            const double f1 = (k == s) ? __ldg(d.sq2 + nk) : __ldg(d.sq + nk) * __ldg(d.sq + ns);
            double r1[M], r2[M];
#pragma unroll
            for (int j = 0; j < M; ++j) {
                const int mj = n[j] - (j == k) - (j == s);
                r1[j] = __ldg(d.sq + mj + 1);
                r2[j] = __ldg(d.sq2 + mj + 2);
            }
            const double2* vrow = sV + mcb_pair_index(M, k, s) * P;
            double wr = 0.0, wi = 0.0;
            int c = 0;
#pragma unroll
            for (int q = 0; q < M; ++q) {
#pragma unroll
                for (int l = q; l < M; ++l, ++c) {
                    const double2 z = __ldg(p.C + MCB_CHK(d, tcur[c], d.nc, 601));
                    const double f2 = (q == l) ? r2[q] : r1[q] * r1[l];
                    const double2 v = vrow[c];
                    const double zr = f2 * z.x, zi = f2 * z.y;
                    wr = fma(v.x, zr, wr); wr = fma(-v.y, zi, wr);
                    wi = fma(v.x, zi, wi); wi = fma(v.y, zr, wi);
                }
            }
            re = fma(f1, wr, re); im = fma(f1, wi, im);
            if (PREFETCH) {
#pragma unroll
                for (int cc = 0; cc < P; ++cc) tcur[cc] = tnext[PREFETCH ? cc : 0];
            }
            line += P;
        }
    }
    p.HC[g] = make_double2(re, im);
}

// Many orbitals (P > 15, where a thread cannot keep a stride in registers): a group of GS lanes per output configuration g walks
// the line stride by stride (coalesced map reads, one gather per lane and stride, partial sums added by shuffles);
// M2C_GTHREADS threads per persistent block share one copy of Vp.  Shared memory:
// Vp [P*P] complex, the sqrt tables, per group the occupations n[M] and the list of its allowed removal pairs.
#define M2C_GTHREADS 256
template <int M, int GS>
__global__ void __launch_bounds__(M2C_GTHREADS) k_hc_maps2c_group(const M2cArgs p)
{
    constexpr int P = M * (M + 1) / 2;
    constexpr int GROUPS = M2C_GTHREADS / GS;
    constexpr int NE = (P + GS - 1) / GS;                                // entries of a stride per lane
    extern __shared__ double2 m2c_smem[];
    double2* sV = m2c_smem;                                              // [P*P]
    double* sSq = reinterpret_cast<double*>(sV + P * P);                 // [N+3] sqrt(j)
    double* sSq2 = sSq + (p.d.N + 3);                                    // [N+3] sqrt(j (j-1))
    int* sN = reinterpret_cast<int*>(sSq2 + (p.d.N + 3));                // [GROUPS][M]
    unsigned short* sList = reinterpret_cast<unsigned short*>(sN + GROUPS * M);   // [GROUPS][P]: (k << 8) | s of the allowed removals
    const McbDev& d = p.d;
    for (int i = threadIdx.x; i < P * P; i += M2C_GTHREADS) sV[i] = p.Vp[i];
    for (int i = threadIdx.x; i < d.N + 3; i += M2C_GTHREADS) { sSq[i] = d.sq[i]; sSq2[i] = d.sq2[i]; }
    const int grp = threadIdx.x / GS, lane = threadIdx.x % GS;
    __syncthreads();                                                     // Vp and the tables are staged ONCE per (persistent) block
    const int* n = sN + grp * M;
    const unsigned short* lst = sList + grp * P;
    const long long per_round = (long long)gridDim.x * GROUPS;
#pragma unroll 1
    for (long long g_base = (long long)blockIdx.x * GROUPS; g_base < d.nc; g_base += per_round) {
    const long long g_ll = g_base + grp;
    // (every group of a warp makes the same number of rounds: the warp-level barriers below are convergent)
    const bool live = g_ll < d.nc;
    const int g = live ? (int)g_ll : 0;
    __syncwarp();                                                        // the previous round is done with n and the list
    if (lane < M) sN[grp * M + lane] = (int)__ldg(p.fock.occ + (long long)lane * p.fock.ld + g);
    __syncwarp();
    // the allowed removals of this line, in the paper's order (every lane walks the same short loop; lane 0 writes the list)
    int cnt = 0;
    {
        unsigned short* lstw = sList + grp * P;
        for (int k = 0; k < M; ++k) {
            if (n[k] < 1) continue;
            for (int s = k; s < M; ++s) {
                if ((k == s) ? (n[k] < 2) : (n[s] < 1)) continue;
                if (lane == 0) lstw[cnt] = (unsigned short)((k << 8) | s);
                ++cnt;
            }
        }
        if (!live) cnt = 0;
    }
    __syncwarp();
    // this lane's replacement pairs (q <= l) of a stride, c = lane + GS e, with everything of (q, l) that does not depend on
    // the removal: the occupations and the three possible factors sqrt(n + 1 - d), d = 0, 1, 2 particles removed from the orbital
    int cq[NE], cl[NE];
    double fq[NE][3], fl[NE][3];
#pragma unroll
    for (int e = 0; e < NE; ++e) {
        int c = lane + GS * e, q = 0, len = M;
        if (c >= P) c = 0;
        while (c >= len) { c -= len; --len; ++q; }
        const int l = q + c;
        cq[e] = q; cl[e] = l;
        const int nq = n[q], nl = n[l];
        if (q == l) {                                                    // sqrt((m_q + 1)(m_q + 2)), m_q = n_q - d
            fq[e][0] = sSq2[nq + 2]; fq[e][1] = sSq2[nq + 1]; fq[e][2] = sSq2[nq > 0 ? nq : 0];
            fl[e][0] = 1.0; fl[e][1] = 1.0; fl[e][2] = 1.0;
        } else {                                                         // sqrt(m_q + 1) sqrt(m_l + 1)
            fq[e][0] = sSq[nq + 1]; fq[e][1] = sSq[nq]; fq[e][2] = sSq[nq > 0 ? nq - 1 : 0];
            fl[e][0] = sSq[nl + 1]; fl[e][1] = sSq[nl]; fl[e][2] = sSq[nl > 0 ? nl - 1 : 0];
        }
    }
    double re = 0.0, im = 0.0;
    const int* row = p.entries + (live ? p.soff[g] : 0) * (long long)P + lane;
    // software pipeline over the strides of the line: map entries are loaded two strides ahead of their gathers, the gathers
    // of C one stride ahead of their use -- neither a gather nor an FMA waits for the load in front of it.  Two target
    // buffers and two value buffers alternate (loop unrolled by two: no register moves)
    int tA[NE], tB[NE];
    double2 zA[NE], zB[NE];
    auto load_map = [&](int (&t)[NE], const int r) {
#pragma unroll
        for (int e = 0; e < NE; ++e) t[e] = (r < cnt && lane + GS * e < P) ? __ldcs(row + (long long)r * P + GS * e) : 0;
    };
    auto gather = [&](double2 (&z)[NE], const int (&t)[NE]) {
#pragma unroll
        for (int e = 0; e < NE; ++e) z[e] = __ldg(p.C + MCB_CHK(d, t[e], d.nc, 601));
    };
    auto consume = [&](const int r, const double2 (&z)[NE]) {
        const int ks = lst[r];
        const int ck = ks >> 8, cs = ks & 255;
        const int ca = mcb_pair_index(M, ck, cs);
        const double f1 = (ck == cs) ? sSq2[n[ck]] : sSq[n[ck]] * sSq[n[cs]];
        double wr = 0.0, wi = 0.0;
#pragma unroll
        for (int e = 0; e < NE; ++e) {
            if (lane + GS * e < P) {
                const int q = cq[e], l = cl[e];
                const int dq = (q == ck) + (q == cs), dl = (l == ck) + (l == cs);
                const double f2 = (dq == 0 ? fq[e][0] : (dq == 1 ? fq[e][1] : fq[e][2])) * (dl == 0 ? fl[e][0] : (dl == 1 ? fl[e][1] : fl[e][2]));
                const double2 v = sV[ca * P + lane + GS * e];
                const double zr = f2 * z[e].x, zi = f2 * z[e].y;
                wr = fma(v.x, zr, wr); wr = fma(-v.y, zi, wr);
                wi = fma(v.x, zi, wi); wi = fma(v.y, zr, wi);
            }
        }
        re = fma(f1, wr, re); im = fma(f1, wi, im);
    };
    // state at the top of the loop: zA = values of stride r, tB = targets of stride r + 1, tA = targets of stride r + 2
    load_map(tA, 0); load_map(tB, 1);
    if (cnt > 0) gather(zA, tA);
    load_map(tA, 2);
#pragma unroll 1
    for (int r = 0; r < cnt; r += 2) {
        if (r + 1 < cnt) gather(zB, tB);
        load_map(tB, r + 3);
        consume(r, zA);
        if (r + 1 < cnt) {
            if (r + 2 < cnt) gather(zA, tA);
            load_map(tA, r + 4);
            consume(r + 1, zB);
        }
    }
    // sum over the lanes of the group (fixed order)
#pragma unroll
    for (int o = GS / 2; o >= 1; o >>= 1) {
        re += __shfl_xor_sync(0xffffffffu, re, o);
        im += __shfl_xor_sync(0xffffffffu, im, o);
    }
    if (live && lane == 0) p.HC[g] = make_double2(re, im);
    }
}

// =========================================================================================================
// host
// =========================================================================================================
static long long m2c_nblocks(const mcb_space* sp) { return (sp->nc + M2C_BLOCK - 1) / M2C_BLOCK; }
static long long m2c_soff_bytes(const mcb_space* sp) { return mcb_round_up((sp->nc + 1) * (long long)sizeof(long long), 256); }
static long long m2c_bsum_bytes(const mcb_space* sp) { return mcb_round_up((m2c_nblocks(sp) + 1) * (long long)sizeof(long long), 256); }

long long mcb_map2c_bytes(const mcb_space* sp)
{
    // sum over configurations of the allowed removals = P nc2 (every (intermediate, pair) is reached exactly once)
    const long long strides = (long long)sp->P * sp->nc2;
    return m2c_soff_bytes(sp) + m2c_bsum_bytes(sp) + mcb_round_up(strides * sp->P * (long long)sizeof(int), 256);
}

static int m2c_pair_tables(mcb_space* sp)
{
    if (sp->d_pair_ks) return MCB_OK;
    const int P = sp->P, M = sp->M;
    unsigned short* h = (unsigned short*)malloc(sizeof(unsigned short) * 2 * (size_t)P);
    if (!h) return MCB_ENOMEM;
    int a = 0;
    for (int k = 0; k < M; ++k)
        for (int s = k; s < M; ++s, ++a) { h[a] = (unsigned short)k; h[P + a] = (unsigned short)s; }
    cudaError_t e = cudaMalloc(&sp->d_pair_ks, sizeof(unsigned short) * 2 * (size_t)P);
    if (e == cudaSuccess) e = cudaMemcpy(sp->d_pair_ks, h, sizeof(unsigned short) * 2 * (size_t)P, cudaMemcpyHostToDevice);
    free(h);
    if (e != cudaSuccess) { if (sp->d_pair_ks) { cudaFree(sp->d_pair_ks); sp->d_pair_ks = NULL; } return mcb_set_cuda_error(e); }
    return MCB_OK;
}

int mcb_pair_tables(mcb_space* sp) { return m2c_pair_tables(sp); }

int mcb_launch_map2c(mcb_space* sp, void* d_buf, cudaStream_t st)
{
    if (!sp->d_fock) return MCB_ENOTREADY;                               // the counts come from the hashing table
    if (sp->N < 2) return MCB_EUNSUPPORTED;
    { int rc = m2c_pair_tables(sp); if (rc) return rc; }
    long long* soff = (long long*)d_buf;
    long long* bsum = (long long*)((char*)d_buf + m2c_soff_bytes(sp));
    int* entries = (int*)((char*)d_buf + m2c_soff_bytes(sp) + m2c_bsum_bytes(sp));
    const int nb = (int)m2c_nblocks(sp);
    k_m2c_count<<<nb, 256, 0, st>>>(sp->dev, sp->fock.occ, sp->fock.ld, bsum);
    MCB_CHECK_LAUNCH();
    k_m2c_scan<<<1, 1024, 0, st>>>(bsum, nb, bsum + nb);
    MCB_CHECK_LAUNCH();
    k_m2c_offsets<<<nb, 256, 0, st>>>(sp->dev, sp->fock.occ, sp->fock.ld, bsum, bsum + nb, soff);
    MCB_CHECK_LAUNCH();
    {
        const int threads = 128;
        const unsigned blocks = (unsigned)((sp->nc + threads - 1) / threads);
        // two blocks per SM (shared memory as the occupancy knob): the partly written sectors of the resident threads' lines
        // must stay in L2 until the next strides complete them (measured at configs[2]: 6.0 ms with 16 blocks per SM, 4.2 with
        // 4, 3.0 with 2, 3.6 with 1; configs[4]: 77 / 70 / 60 / 52 ms)
#ifndef M2C_FILL_BLOCKS_SM
#define M2C_FILL_BLOCKS_SM 2
#endif
        const size_t pad = ((size_t)(220 * 1024) / M2C_FILL_BLOCKS_SM) & ~(size_t)15;
        MCB_DISPATCH_M(sp->M, (cudaFuncSetAttribute(k_m2c_fill<MT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pad)));
        MCB_DISPATCH_M(sp->M, (k_m2c_fill<MT><<<blocks, threads, pad, st>>>(sp->dev, sp->fock.occ, sp->fock.ld, soff, entries)));
    }
    MCB_CHECK_LAUNCH();
    sp->d_map2c = d_buf;
    return MCB_OK;
}

// logical export for the parity tests: stride offsets of configurations b0 .. b0 + count (count + 1 values, absolute) and
// the entries of those lines, in the paper's order
int mcb_map2c_export_impl(const mcb_space* sp, long long b0, long long count, long long* host_soff, int* host_entries, long long capacity)
{
    if (!sp->d_map2c) return MCB_ENOTREADY;
    const long long* soff = (const long long*)sp->d_map2c;
    const int* entries = (const int*)((const char*)sp->d_map2c + m2c_soff_bytes(sp) + m2c_bsum_bytes(sp));
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(host_soff, soff + b0, sizeof(long long) * (size_t)(count + 1), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return mcb_set_cuda_error(e);
    const long long n_entries = (host_soff[count] - host_soff[0]) * sp->P;
    if (n_entries > capacity) return MCB_ENOMEM;
    if (n_entries > 0) {
        e = cudaMemcpy(host_entries, entries + host_soff[0] * sp->P, sizeof(int) * (size_t)n_entries, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return mcb_set_cuda_error(e);
    }
    return MCB_OK;
}

template <int M>
static int launch_maps2c_t(mcb_space* sp, const M2cArgs& a, cudaStream_t st)
{
    constexpr int P = M * (M + 1) / 2;
    const size_t smem = sizeof(double2) * P * P;
    if (!(sp->attr_set & (1u << 8))) {
        MCB_CUDA(cudaFuncSetAttribute(k_hc_maps2c<M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        sp->attr_set |= 1u << 8;
    }
    const unsigned blocks = (unsigned)((sp->nc + M2C_THREADS - 1) / M2C_THREADS);
    k_hc_maps2c<M><<<blocks, M2C_THREADS, smem, st>>>(a);
    MCB_CHECK_LAUNCH();
    return MCB_OK;
}

template <int M, int GS>
static int launch_maps2c_group(mcb_space* sp, const M2cArgs& a, cudaStream_t st)
{
    constexpr int P = M * (M + 1) / 2;
    constexpr int GROUPS = M2C_GTHREADS / GS;
    const size_t smem = sizeof(double2) * P * P + 2 * sizeof(double) * (size_t)(sp->N + 3) + sizeof(int) * GROUPS * M
                        + sizeof(unsigned short) * GROUPS * P + 16;
    if (smem > 227 * 1024) return MCB_EUNSUPPORTED;
    if (sp->maps2c_grid == 0) {                                          // once per space: smem depends on (N, M) only
        MCB_CUDA(cudaFuncSetAttribute(k_hc_maps2c_group<M, GS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int per_sm = 0, sms = 0;
        MCB_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_hc_maps2c_group<M, GS>, M2C_GTHREADS, smem));
        MCB_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, sp->device));
        if (per_sm < 1) return MCB_EUNSUPPORTED;
        sp->maps2c_grid = (long long)per_sm * sms;
    }
    long long blocks = (sp->nc + GROUPS - 1) / GROUPS;
    if (blocks > sp->maps2c_grid) blocks = sp->maps2c_grid;              // persistent: Vp is staged once per block
    k_hc_maps2c_group<M, GS><<<(unsigned)blocks, M2C_GTHREADS, smem, st>>>(a);
    MCB_CHECK_LAUNCH();
    return MCB_OK;
}

int mcb_launch_maps2c(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_C, mcb_c128* d_HC, cudaStream_t st)
{
    const int P = sp->P, M = sp->M;
    const size_t pp = (size_t)P * P;
    if (sizeof(double) * 4 * pp > sp->coef_bytes) return MCB_ENOMEM;
    if (mcb_coef_stale(sp)) {
        double* h = (double*)sp->h_coef;
        double* vr = h + 2 * pp;
        double* vi = vr + pp;
        mcb_pack_pairs(sp->N, M, T, V, true, vr, vi);                    // T folded in: no single-jump map needed
        for (size_t i = 0; i < pp; ++i) { h[2 * i] = vr[i]; h[2 * i + 1] = vi[i]; }
        { int rc = mcb_coef_upload(sp, h, sizeof(double) * 2 * pp, st); if (rc) return rc; }
        mcb_coef_staged(sp);
    }
    M2cArgs a;
    a.d = sp->dev; a.fock = sp->fock;
    a.C = (const double2*)d_C; a.HC = (double2*)d_HC; a.Vp = (const double2*)sp->d_coef;
    a.soff = (const long long*)sp->d_map2c;
    a.entries = (const int*)((const char*)sp->d_map2c + m2c_soff_bytes(sp) + m2c_bsum_bytes(sp));
    a.nstrides = (long long)sp->P * sp->nc2;
    { int rc = mcb_tick(sp, 0, st); if (rc) return rc; }
    int rc = MCB_EUNSUPPORTED;
    switch (M) {
    case 1: rc = launch_maps2c_t<1>(sp, a, st); break;                   // one orbital: nc = 1, one stride of one target
    case 2: rc = launch_maps2c_t<2>(sp, a, st); break;
    case 3: rc = launch_maps2c_t<3>(sp, a, st); break;
    case 4: rc = launch_maps2c_t<4>(sp, a, st); break;
    case 5: rc = launch_maps2c_t<5>(sp, a, st); break;
    case 6: rc = launch_maps2c_group<6, 32>(sp, a, st); break;
    case 7: rc = launch_maps2c_group<7, 32>(sp, a, st); break;
    case 8: rc = launch_maps2c_group<8, 32>(sp, a, st); break;
    case 9: rc = launch_maps2c_group<9, 32>(sp, a, st); break;
    case 10: rc = launch_maps2c_group<10, 32>(sp, a, st); break;
    case 11: rc = launch_maps2c_group<11, 32>(sp, a, st); break;
    case 12: rc = launch_maps2c_group<12, 32>(sp, a, st); break;
    default: break;
    }
    if (rc != MCB_OK) return rc;
    { int rc2 = mcb_tick(sp, 1, st); if (rc2) return rc2; }
    mcb_tick_done(sp, 1);
    sp->last_launches = 1;
    return MCB_OK;
}
