// mcb_apply_runs.cu -- MCB_RUNS mode of hc_apply (Eq. 12-13) for few orbitals (2 <= M <= 5).
//
// Same factorisation through the (N-2)-particle space as MCB_GEMM (mcb_apply_gemm.cu),
//     H = sum_m sum_{a=(k<=s)} sum_{c=(q<=l)} |m+e_k+e_s> F(m,a) Vp[a][c] F(m,c) <m+e_q+e_l|   (T folded into Vp),
// laid out for the "few orbitals, many particles" shape (M = 3..5, N = 100..1000), where the
// index order has long runs (only n_0, n_1 change inside a run; run length ~ (N+M-1)/(M-1)):
//
// ONE persistent kernel per apply, k_hc2_runs<M>, with two roles.
//   CONTRACTING warps take short segments of consecutive intermediates in index order from a global ticket and walk
//     them in chunks of 32, as one software pipeline that never drains, three deep:
//       A  (lane = intermediate)  occupations of chunk ch+2 are loaded; for chunk ch+1 the index arithmetic
//          (mcb_device.cuh) runs and the P targets of C are gathered with cp.async straight into the warp's
//          shared-memory stage Z[c][m]; the factors F(m,c) and the output indices go beside them;
//       B  (tensor path)          for chunk ch, four 8-intermediate blocks: A-fragment = F(m,c) * Z[c][m] read from
//          the stage, B-fragment = the packed coefficients embedded as a real (2P x 2P) matrix, STATIONARY in
//          registers; mma.sync.m8n8k4.f64 (SASS DMMA) accumulates W'[a][m], which is scaled by F(m,a) and staged
//          in shared memory;
//       C  (lane = intermediate)  in-run pre-summation and store.  Orbitals 0 and 1 only move a configuration
//          inside its run (index +-1), so the removal pairs fall into classes kappa = (the part of e_k+e_s on
//          orbitals >= 2):
//              {}      : (0,0) (0,1) (1,1)          -> outputs g0, g0+1, g0+2 with g0 = index(m + 2 e_0)
//              {h}     : (0,h) (1,h)                -> outputs gh, gh+1       with gh = index(m + e_0 + e_h)
//              {h,h'}  : (h,h')                     -> output  index(m + e_h + e_h')
//          and the contributions of one class to one output come from up to three NEIGHBOURING intermediates of
//          the same run -- neighbouring slots of the stage.  They are summed and written once into a plane
//          Hp[kappa][g] indexed by the OUTPUT configuration (NCLS = 1 + (M-2) + (M-2)(M-1)/2 planes instead of
//          P), each (kappa, g) slot by exactly one thread: no atomics.
//   SUMMING warps (one per CTA, and every contracting warp once the tickets run out) take tiles of outputs in index
//     order: HC[g] = sum over the classes allowed at g of Hp[kappa][g], a coalesced stream that trails the
//     contraction behind per-segment release/acquire flags (run_sum_tiles).
#include <string.h>
#include "mcb_device.cuh"

#ifndef RUNS_CHUNKS
#define RUNS_CHUNKS 16
#endif
__host__ __device__ constexpr int rdiv(int a, int b) { return (a + b - 1) / b; }

template <int M> struct RunCfg {
    static constexpr int P = M * (M + 1) / 2;
    static constexpr int NH = M - 2;                               // orbitals that leave the run
    static constexpr int NCLS = 1 + NH + NH * (NH + 1) / 2;        // classes = planes
    static constexpr int NK = rdiv(2 * P, 4);                      // k-steps (contraction over (c, re|im))
    static constexpr int NB = rdiv(2 * P, 8);                      // 8-column blocks of outputs (a, re|im)
    static constexpr int CHUNKS = RUNS_CHUNKS;                              // 32-wide chunks per segment (one ticket)
    static constexpr int SEG = CHUNKS * 32 - 2;                    // intermediates OWNED per segment (2 halo lanes)
    // per-warp shared memory, two stages of
    //   [2 carry slots][ Z / W' : P rows x ZLD double2 ][ F : P rows x FLD double ][ META : MROWS rows x 32 int ]
    // Z[c][m] receives the gathered C values of chunk ch; once the DMMAs of the chunk are done the same rows hold
    // W'[a][m] for phase C.  Slots 32..35 of a row are padding (36 % 8 == 4 makes the A-fragment reads conflict
    // free); slots 34, 35 of row a - 1 (the two slots in FRONT of row a) carry W'[a] of lanes 30, 31 of the
    // previous chunk -- cp.async never touches them, so they are written into the stage that is being filled.
    static constexpr int ZLD = 36;
    static constexpr int FLD = 40;                                 // doubles per row of F
    static constexpr int MROWS = NCLS + 1;                         // int rows of META: output index per class, flags
    static constexpr int STAGES = 2;
    static constexpr size_t HEAD_BYTES = 32;
    static constexpr size_t Z_BYTES = (size_t)P * ZLD * 16;
    static constexpr size_t F_BYTES = (size_t)P * FLD * 8;
    static constexpr size_t META_BYTES = (size_t)MROWS * 32 * 4;
    static constexpr size_t STAGE_BYTES = HEAD_BYTES + Z_BYTES + F_BYTES + META_BYTES;
    static constexpr size_t WARP_BYTES = STAGES * STAGE_BYTES;
    // warps per CTA / CTAs per SM: as many warps as the 227 KB hold, in two CTAs
    static constexpr int WARPS_SM = (int)((227 * 1024 - 2 * 1024) / WARP_BYTES);
    static constexpr int WARPS = WARPS_SM / 2 > 8 ? 8 : WARPS_SM / 2;
    static constexpr int THREADS = (WARPS + 1) * 32;               // + one warp per CTA that only sums
#ifndef RUNS_SUM_TILE
#define RUNS_SUM_TILE 1024
#endif
    static constexpr int SUM_TILE = RUNS_SUM_TILE;                 // outputs per sum ticket
    static constexpr int SUM_U = (NCLS <= 6) ? 4 : 2;                  // outputs in flight per lane
    static constexpr size_t SMEM = WARPS * WARP_BYTES;
    static constexpr int MINB = 2;
    static_assert(STAGE_BYTES % 16 == 0 && Z_BYTES % 16 == 0 && F_BYTES % 16 == 0, "alignment");
    static_assert(WARPS >= 1, "shared memory");
};

// Coefficient matrix of the embedded real product, B[kappa][n] with kappa = 2 c + (re|im of the gathered value),
// n = 2 a + (re|im of the result):   W.re = sum Vr z.re - Vi z.im,   W.im = sum Vi z.re + Vr z.im
template <int M> struct RunCoef { double b[RunCfg<M>::NK * 4][RunCfg<M>::NB * 8]; };     // T folded in, zero padded

struct RunArgs {
    McbDev d;
    McbFockView fock;
    const double2* C;
    double2* HC;
    double2* Hp;               // [NCLS][ldp]
    long long ldp;
    int nseg;                  // warp segments of the contraction
    int ntile;                 // output tiles of the sum (SUM_TILE outputs each)
    int* flags;                // [nseg] segment s has been contracted and its class planes are visible
    int* tickets;              // [0] next segment, [1] next output tile, [2] verified prefix of flags,
                               // [3] elements of C that have arrived (pipelined host apply), [4] error word, [5..7] pad
    const int* c_avail;        // pipelined host apply: number of leading elements of C that have arrived (NULL: all)
};

#define RUNS_NTICKETS 8

__device__ __forceinline__ int run_cls_single(int h) { return 1 + (h - 2); }
template <int M> __device__ __forceinline__ constexpr int run_cls_pair(int h, int h2)
{
    // pair index over the NH high orbitals, (h-2) <= (h2-2)
    return 1 + (M - 2) + mcb_pair_index(M - 2, h - 2, h2 - 2);
}

__device__ __forceinline__ void run_dmma884(double& c0, double& c1, const double a, const double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// ---- cp.async (LDGSTS): 16-byte global -> shared copies that do not hold a register while in flight ----------
__device__ __forceinline__ void cp_async16(double2* smem_dst, const double2* gsrc, bool valid)
{
    const unsigned dst = (unsigned)__cvta_generic_to_shared(smem_dst);
    const int bytes = valid ? 16 : 0;                                   // 0 -> the slot is zero-filled
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(gsrc), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// occupations of intermediate m from the hashing table (zeros outside [0, nc2))
template <int M>
__device__ __forceinline__ void run_load_occ(const RunArgs& p, const int m, int (&occ)[M])
{
    const bool valid = m >= 0 && m < p.d.nc2;
#pragma unroll
    for (int j = 0; j < M; ++j) occ[j] = valid ? (int)__ldg(p.fock.occ2 + (long long)j * p.fock.ld2 + m) : 0;
}

// Phase A for one intermediate (this lane's slot of the stage): index arithmetic, asynchronous gather of the P
// targets of C, factors F(m,c) = sqrt((m_q+1)(m_l+1+[q==l])), output indices and flags.
template <int M>
__device__ __forceinline__ void run_prefetch(const RunArgs& p, const int m, const int (&occ)[M], const int seg0, const int seg_end,
                                             unsigned char* __restrict__ stage, const int lane)
{
    using Cfg = RunCfg<M>;
    const McbDev& d = p.d;
    double2* const Z = reinterpret_cast<double2*>(stage + Cfg::HEAD_BYTES) + lane;
    double* const F = reinterpret_cast<double*>(stage + Cfg::HEAD_BYTES + Cfg::Z_BYTES) + lane;
    int* const META = reinterpret_cast<int*>(stage + Cfg::HEAD_BYTES + Cfg::Z_BYTES + Cfg::F_BYTES) + lane;
    const bool valid = m >= 0 && m < d.nc2;
    const bool own = valid && m >= seg0 && m < seg_end;
    int X[M], Y[M], mj0 = 0, mj1 = 0;
    double r1[M], r2[M];
    {
        int A1[M], A2[M];
        int run = 0, x = 0, tot1 = 0;
#pragma unroll
        for (int j = 0; j < M; ++j) {
            const int nj = occ[j];
            if (j == 0) mj0 = nj;
            if (j == 1) mj1 = nj;
            run += nj;
            r1[j] = __ldg(d.sq + nj + 1);
            r2[j] = __ldg(d.sq2 + nj + 2);
            X[j] = x;
            if (j == 0) {
                // G[0][s] = binom(s, 1) = s: no look-up
                A1[0] = run + 1; A2[0] = run + 2;
                x += -1; tot1 += A1[0];
            } else if (j <= M - 2) {
                const int a0 = mcb_ldG(d.G, d.ldg, j, run);
                A1[j] = mcb_ldG(d.G, d.ldg, j, run + 1);
                A2[j] = mcb_ldG(d.G, d.ldg, j, run + 2);
                x += a0 - A1[j]; tot1 += A1[j];
            } else { A1[j] = 0; A2[j] = 0; }
        }
        int pre = tot1, suf = 0;
#pragma unroll
        for (int l = M - 1; l >= 0; --l) { pre -= A1[l]; suf += A2[l]; Y[l] = pre + suf; }
    }
    const int base = d.nc - 1;
    {
        int c = 0;
#pragma unroll
        for (int q = 0; q < M; ++q) {
#pragma unroll
            for (int l = q; l < M; ++l, ++c) {
                cp_async16(Z + c * Cfg::ZLD, p.C + (valid ? MCB_CHK(d, base - X[q] - Y[l], d.nc, 401) : 0), valid);
                F[c * Cfg::FLD] = (q == l) ? r2[q] : r1[q] * r1[l];
            }
        }
    }
    META[0] = valid ? (int)MCB_CHK(d, base - X[0] - Y[0], d.nc, 402) : 0;
#pragma unroll
    for (int h = 2; h < M; ++h) {
        META[run_cls_single(h) * 32] = valid ? (int)MCB_CHK(d, base - X[0] - Y[h], d.nc, 403) : 0;
#pragma unroll
        for (int h2 = h; h2 < M; ++h2) META[run_cls_pair<M>(h, h2) * 32] = valid ? (int)MCB_CHK(d, base - X[h] - Y[h2], d.nc, 404) : 0;
    }
    META[Cfg::NCLS * 32] = (own ? 1 : 0) | (mj0 == 0 ? 2 : 0) | (mj1 << 2);
}

__device__ __forceinline__ void cadd(double2& o, const double2 w) { o.x += w.x; o.y += w.y; }

__device__ __forceinline__ int run_ticket(int* ctr, const int lane)
{
    int t = 0;
    if (lane == 0) t = atomicAdd(ctr, 1);
    return __shfl_sync(0xffffffffu, t, 0);
}

// HC[g] = sum over the classes allowed at g of Hp[kappa][g], for output tiles taken in index order.  A tile whose
// largest top occupation n_{M-1} is j needs every intermediate with m_{M-1} <= j, a PREFIX of the intermediate
// order (nc2 - N_c(N-3-j, M) of them): the warp waits until the segments of that prefix are flagged.  The
// contraction never waits for anything, so this cannot deadlock; it trails the contraction closely enough for
// the class planes to be read from L2.
// Memory model: a producer publishes a segment with st.release.gpu after a __syncwarp; the probes here are strong
// (volatile) loads followed by a gpu-scope fence before the planes are read; the shared verified-prefix watermark is
// published after a fence and read with a strong load followed by the same fence (release/acquire by fence cumulativity).
template <int M>
__device__ __forceinline__ void run_sum_tiles(const RunArgs& p, const int lane)
{
    using Cfg = RunCfg<M>;
    const McbDev& d = p.d;
    int wm = 0;                                                          // segments < wm are known to be done
    for (;;) {
        const int t = run_ticket(p.tickets + 1, lane);
        if (t >= p.ntile) break;
#ifdef RUNS_DEBUG_LAG
        if (lane == 0) { const int lagk = (int)((((long long)*reinterpret_cast<volatile int*>(p.tickets)) * Cfg::SEG - (long long)t * Cfg::SUM_TILE) >> 10); atomicMax(p.tickets + 5, lagk); }
#endif
        const int g0 = t * Cfg::SUM_TILE;
        const int g1 = min(g0 + Cfg::SUM_TILE, d.nc);
        const int jmax = (int)__ldg(p.fock.occ + (long long)(M - 1) * p.fock.ld + (g1 - 1));
        const int tt = max(d.N - 2 - jmax, 0);
        const int need_int = d.nc2 - mcb_ldG(d.G, d.ldg, M - 2, tt);     // G[M-2][t] = N_c(t - 1, M)
        const int need_seg = (need_int + Cfg::SEG - 1) / Cfg::SEG;
        if (wm < need_seg) {
            wm = max(wm, *reinterpret_cast<volatile int*>(p.tickets + 2));          // what other warps have verified
            const int wm_in = wm;
            unsigned backoff = 256;
            while (wm < need_seg) {
                // wait (one lane, one strong load per probe, exponential back-off) until the first unverified segment is flagged
                for (;;) {
                    int f0 = 0;
                    if (lane == 0) asm volatile("ld.volatile.global.s32 %0, [%1];" : "=r"(f0) : "l"(p.flags + wm) : "memory");
                    f0 = __shfl_sync(0xffffffffu, f0, 0);
                    if (f0 != 0) break;
                    __nanosleep(backoff);
                    if (backoff < 4096) backoff *= 2;
                }
                // then sweep 128 flags per round trip; indices outside [wm, need_seg) count as set
                for (;;) {
                    const int a = wm & ~127;
                    int4 f4;
                    asm volatile("ld.volatile.global.v4.s32 {%0,%1,%2,%3}, [%4];"
                                 : "=r"(f4.x), "=r"(f4.y), "=r"(f4.z), "=r"(f4.w) : "l"(reinterpret_cast<const int4*>(p.flags + a) + lane) : "memory");
                    const int f[4] = {f4.x, f4.y, f4.z, f4.w};
                    int first_unset = 4;
#pragma unroll
                    for (int i = 3; i >= 0; --i) {
                        const int idx = a + 4 * lane + i;
                        if (idx >= wm && idx < need_seg && f[i] == 0) first_unset = i;
                    }
                    const unsigned ball = __ballot_sync(0xffffffffu, first_unset < 4);
                    if (ball == 0u) { wm = a + 128; if (wm >= need_seg) break; }
                    else {
                        const int src = __ffs(ball) - 1;
                        wm = a + 4 * src + __shfl_sync(0xffffffffu, first_unset, src);
                        break;
                    }
                }
            }
            wm = min(wm, need_seg);
            __threadfence();                                             // flags observed -> before the watermark is published
            if (lane == 0 && wm > wm_in) atomicMax(p.tickets + 2, wm);
        }
        __threadfence();
        // rounds of 32 * SUM_U outputs, software-pipelined: the occupations of round r + 1 are loaded before the class-plane
        // loads of round r are issued, so a round costs one memory latency instead of two
        int nn[Cfg::SUM_U][M];
#pragma unroll
        for (int u = 0; u < Cfg::SUM_U; ++u) {
            const int g = g0 + u * 32 + lane;
#pragma unroll
            for (int j = 0; j < M; ++j) nn[u][j] = g < g1 ? (int)__ldg(p.fock.occ + (long long)j * p.fock.ld + g) : 0;
        }
#pragma unroll 1
        for (int gb = g0; gb < g1; gb += 32 * Cfg::SUM_U) {
            int n[Cfg::SUM_U][M];
#pragma unroll
            for (int u = 0; u < Cfg::SUM_U; ++u) {
                const int gnext = gb + 32 * Cfg::SUM_U + u * 32 + lane;
#pragma unroll
                for (int j = 0; j < M; ++j) {
                    n[u][j] = nn[u][j];
                    nn[u][j] = gnext < g1 ? (int)__ldg(p.fock.occ + (long long)j * p.fock.ld + gnext) : 0;
                }
            }
            // all loads of SUM_U outputs are issued before the first add: SUM_U * NCLS 16-byte loads in flight per lane
            double2 w[Cfg::SUM_U][Cfg::NCLS];
#pragma unroll
            for (int u = 0; u < Cfg::SUM_U; ++u) {
                const int g = gb + u * 32 + lane;
                const int in01 = n[u][0] + n[u][1];
                const double2* src = p.Hp + g;
                const double2 zero = make_double2(0.0, 0.0);
                w[u][0] = (in01 >= 2) ? __ldcg(src) : zero;
#pragma unroll
                for (int h = 2; h < M; ++h)
                    w[u][run_cls_single(h)] = (n[u][h] >= 1 && in01 >= 1) ? __ldcg(src + (long long)run_cls_single(h) * p.ldp) : zero;
#pragma unroll
                for (int h = 2; h < M; ++h) {
#pragma unroll
                    for (int h2 = h; h2 < M; ++h2) {
                        const bool ok = (h == h2) ? (n[u][h] >= 2) : (n[u][h] >= 1 && n[u][h2] >= 1);
                        w[u][run_cls_pair<M>(h, h2)] = ok ? __ldcg(src + (long long)run_cls_pair<M>(h, h2) * p.ldp) : zero;
                    }
                }
            }
#pragma unroll
            for (int u = 0; u < Cfg::SUM_U; ++u) {
                const int g = gb + u * 32 + lane;
                double re = 0.0, im = 0.0;
#pragma unroll
                for (int k = 0; k < Cfg::NCLS; ++k) { re += w[u][k].x; im += w[u][k].y; }
                if (g < g1) __stwt(p.HC + g, make_double2(re, im));
            }
        }
    }
}

template <int M>
__global__ void __launch_bounds__(RunCfg<M>::THREADS, RunCfg<M>::MINB)
k_hc2_runs(const RunArgs p, const __grid_constant__ RunCoef<M> coef)
{
    using Cfg = RunCfg<M>;
    constexpr int P = Cfg::P, NK = Cfg::NK, NB = Cfg::NB;
    extern __shared__ __align__(16) unsigned char run_smem[];
    const McbDev& d = p.d;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int grp = lane >> 2, tig = lane & 3;
    if (warp == Cfg::WARPS) { run_sum_tiles<M>(p, lane); return; }       // the summing warp of this CTA
    unsigned char* const wbase = run_smem + (size_t)warp * Cfg::WARP_BYTES;

    // stationary B-fragments: b[ks][nb] = B[4 ks + tig][8 nb + grp]
    double bfrag[NK][NB];
#pragma unroll
    for (int ks = 0; ks < NK; ++ks)
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) bfrag[ks][nb] = coef.b[4 * ks + tig][8 * nb + grp];

    // The warp walks a STREAM of chunks: the chunks of one short segment after the other, segments taken in index
    // order from a global ticket, so that at any moment all warps of the GPU work inside a narrow window of the
    // intermediate order (the class planes they write are still in L2 when the sum reads them) while the software
    // pipeline (occupations of chunk i+2 | gathers of chunk i+1 | DMMAs of chunk i) never drains.
    struct Chunk { int m0, seg0, seg_end, seg; bool valid, last; };
    int gen_seg = 0, gen_ch = 0, gen_nch = 0;                            // generator state: next chunk of the stream
    auto next_chunk = [&](Chunk& c) {
        if (gen_ch == gen_nch) {                                         // segment exhausted: take the next ticket
            gen_seg = run_ticket(p.tickets, lane);
            gen_ch = 0;
            gen_nch = gen_seg < p.nseg ? (min(gen_seg * Cfg::SEG + Cfg::SEG, d.nc2) - (gen_seg * Cfg::SEG - 2) + 31) >> 5 : 0;
            if (p.c_avail != nullptr && gen_nch > 0) {
                // C is still streaming in from the host (mcb_hc_apply_host): an intermediate with top occupation j gathers
                // targets with n_{M-1} <= j + 2 only, i.e. inside the first nc - N_c(N-j-3, M) elements of C
                const int last = min(gen_seg * Cfg::SEG + Cfg::SEG, d.nc2) - 1;
                const int jtop = (int)__ldg(p.fock.occ2 + (long long)(M - 1) * p.fock.ld2 + last);
                const int need = d.nc - mcb_ldG(d.G, d.ldg, M - 2, max(d.N - (jtop + 2), 0));
                int have;
                // bounded: if a piece of C never arrives (a failed copy) the kernel gives up after ~4 s, raises the error
                // word (checked by the host) and runs to completion on whatever is there instead of hanging.  The wait is
                // bounded for the KERNEL, not per segment: once any warp has raised the word, nobody waits again
                for (unsigned spins = 0;; ++spins) {
                    asm volatile("ld.acquire.sys.global.s32 %0, [%1];" : "=r"(have) : "l"(p.c_avail) : "memory");
                    if (have >= need) break;
                    if ((spins & 63u) == 0 && *reinterpret_cast<const volatile int*>(p.tickets + 4) != 0) break;
                    if (spins > (1u << 21)) { if (lane == 0) atomicExch(p.tickets + 4, 1); break; }
                    __nanosleep(2000);
                }
            }
            if (gen_nch == 0) { gen_nch = -1; }                          // no work left, stay exhausted
        }
        c.valid = gen_nch > 0;
        if (!c.valid) { gen_ch = gen_nch = -1; c.m0 = 0; c.seg0 = 0; c.seg_end = 0; c.seg = 0; c.last = false; return; }
        c.seg = gen_seg;
        c.seg0 = gen_seg * Cfg::SEG;
        c.seg_end = min(c.seg0 + Cfg::SEG, d.nc2);
        c.m0 = c.seg0 - 2 + gen_ch * 32;                                 // two halo lanes in front of the segment
        ++gen_ch;
        c.last = gen_ch == gen_nch;
    };
    Chunk c0, c1, c2;
    next_chunk(c0); next_chunk(c1); next_chunk(c2);
    int occ[M];
    int st = 0;
    if (c0.valid) {
        run_load_occ<M>(p, c0.m0 + lane, occ);
        run_prefetch<M>(p, c0.m0 + lane, occ, c0.seg0, c0.seg_end, wbase, lane);
    }
    cp_async_commit();
    if (c1.valid) run_load_occ<M>(p, c1.m0 + lane, occ);

#pragma unroll 1
    while (c0.valid) {
        // ---- phase A: next chunk (its gathers fly under the DMMAs of this one), occupations of the one after ----
        unsigned char* const stage_next = wbase + (st ^ 1) * Cfg::STAGE_BYTES;
        if (c1.valid) run_prefetch<M>(p, c1.m0 + lane, occ, c1.seg0, c1.seg_end, stage_next, lane);
        cp_async_commit();
        if (c2.valid) run_load_occ<M>(p, c2.m0 + lane, occ);
        cp_async_wait<1>();                                              // this lane's gathers of chunk ch have landed
        __syncwarp();                                                    // ... and everybody else's
        unsigned char* const stage = wbase + st * Cfg::STAGE_BYTES;
        const double* Zd = reinterpret_cast<const double*>(stage + Cfg::HEAD_BYTES);                          // [P][ZLD][re|im]
        double2* const W = reinterpret_cast<double2*>(stage + Cfg::HEAD_BYTES);                               // [P][ZLD], after the DMMAs
        const double* F = reinterpret_cast<const double*>(stage + Cfg::HEAD_BYTES + Cfg::Z_BYTES);             // [P][FLD]
        const int* META = reinterpret_cast<const int*>(stage + Cfg::HEAD_BYTES + Cfg::Z_BYTES + Cfg::F_BYTES); // [MROWS][32]

        // ---- phase B: W'[a][m] = F(m,a) sum_c Vp[a][c] F(m,c) Z[c][m]; the four 8-intermediate blocks of the
        //      chunk are in flight together: 4 NB independent DMMA accumulator chains ----
        {
            double acc[4][NB][2];
#pragma unroll
            for (int cb = 0; cb < 4; ++cb)
#pragma unroll
                for (int nb = 0; nb < NB; ++nb) { acc[cb][nb][0] = 0.0; acc[cb][nb][1] = 0.0; }
#pragma unroll
            for (int ks = 0; ks < NK; ++ks) {
                const int c = 2 * ks + (tig >> 1);                       // kappa = 4 ks + tig = 2 c + part
                double a[4];
#pragma unroll
                for (int cb = 0; cb < 4; ++cb) {
                    a[cb] = 0.0;
                    if (2 * ks + 1 < P || c < P)
                        a[cb] = Zd[(c * Cfg::ZLD + cb * 8 + grp) * 2 + (tig & 1)] * F[c * Cfg::FLD + cb * 8 + grp];
                }
#pragma unroll
                for (int cb = 0; cb < 4; ++cb)
#pragma unroll
                    for (int nb = 0; nb < NB; ++nb) run_dmma884(acc[cb][nb][0], acc[cb][nb][1], a[cb], bfrag[ks][nb]);
            }
            __syncwarp();                                                // every lane is done with Z: the rows become W'
#pragma unroll
            for (int cb = 0; cb < 4; ++cb)
#pragma unroll
                for (int nb = 0; nb < NB; ++nb) {
                    const int ar = 4 * nb + tig;                         // this lane holds (re, im) of W'[ar][cb * 8 + grp]
                    if (4 * nb + 3 < P || ar < P) {
                        const double f = F[ar * Cfg::FLD + cb * 8 + grp];
                        W[ar * Cfg::ZLD + ((cb * 8 + grp) ^ ((tig >> 1) << 1))] = make_double2(f * acc[cb][nb][0], f * acc[cb][nb][1]);
                    }
                }
        }
        __syncwarp();

        // ---- phase C: in-run pre-summation (lane = intermediate; slots -1, -2 of lane 0 are the carry slots) and
        //      one store per (class, output) ----
        {
            // row a of W' is stored with bit 1 of the slot flipped when bit 1 of a is set: with the 36-slot row stride this
            // makes the fragment stores of phase B conflict free (rows 4 nb + tig, tig = 0..3, otherwise collide in pairs);
            // the carry slots -1, -2 (in the padding in front of the row) are not swizzled
            auto Wat = [&](const int a, const int back) -> const double2& {
                const int sl = lane - back;
                return W[a * Cfg::ZLD + (sl >= 0 ? (sl ^ (((a >> 1) & 1) << 1)) : sl)];
            };
            const int flags = META[Cfg::NCLS * 32 + lane];
            const bool own = flags & 1, last = flags & 2;
            const int mj1 = flags >> 2;
            constexpr int a00 = mcb_pair_index(M, 0, 0), a01 = mcb_pair_index(M, 0, 1), a11 = mcb_pair_index(M, 1, 1);
            if (own) {
                // class {}: pairs (0,0), (0,1), (1,1)
                double2 o = Wat(a00, 0);
                if (mj1 >= 1) cadd(o, Wat(a01, 1));
                if (mj1 >= 2) cadd(o, Wat(a11, 2));
                double2* dst = p.Hp + META[lane];
                __stcg(dst, o);
                if (last) {
                    double2 e = Wat(a01, 0);
                    if (mj1 >= 1) cadd(e, Wat(a11, 1));
                    __stcg(dst + 1, e);
                    __stcg(dst + 2, Wat(a11, 0));
                }
                // class {h}: pairs (0,h), (1,h)
#pragma unroll
                for (int h = 2; h < M; ++h) {
                    const int a0 = mcb_pair_index(M, 0, h), a1 = mcb_pair_index(M, 1, h);
                    double2 oh = Wat(a0, 0);
                    if (mj1 >= 1) cadd(oh, Wat(a1, 1));
                    double2* dh = p.Hp + (long long)run_cls_single(h) * p.ldp + META[run_cls_single(h) * 32 + lane];
                    __stcg(dh, oh);
                    if (last) __stcg(dh + 1, Wat(a1, 0));
                }
                // class {h,h'}: one pair, one output
#pragma unroll
                for (int h = 2; h < M; ++h) {
#pragma unroll
                    for (int h2 = h; h2 < M; ++h2) {
                        const int cls = run_cls_pair<M>(h, h2);
                        __stcg(p.Hp + (long long)cls * p.ldp + META[cls * 32 + lane], Wat(mcb_pair_index(M, h, h2), 0));
                    }
                }
            }
            if (lane >= 30) {                                            // carry the rows that neighbours read
                double2* Wn = reinterpret_cast<double2*>(stage_next + Cfg::HEAD_BYTES) + lane - 32;
                Wn[a01 * Cfg::ZLD] = Wat(a01, 0);
                Wn[a11 * Cfg::ZLD] = Wat(a11, 0);
#pragma unroll
                for (int h = 2; h < M; ++h) Wn[mcb_pair_index(M, 1, h) * Cfg::ZLD] = Wat(mcb_pair_index(M, 1, h), 0);
            }
            __syncwarp();                                                // W' of this stage may now be overwritten
        }
        if (c0.last) {                                                   // publish: the class-plane stores of the segment
            __syncwarp();                                                // are visible before its flag: the barrier orders
            if (lane == 0)                                               // the warp's stores before lane 0's release store
                asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p.flags + c0.seg), "r"(1) : "memory");
        }
        c0 = c1; c1 = c2; next_chunk(c2);
        st ^= 1;
    }
    run_sum_tiles<M>(p, lane);                                           // no segment left: help with the sum
}

// =========================================================================================================
// host
// =========================================================================================================
static long long runs_ldp(const mcb_space* sp) { return mcb_round_up(sp->nc, 128); }
// tickets + segment flags; sized for the shortest segment any M uses
static long long runs_sync_bytes(const mcb_space* sp)
{
    const long long nseg = (sp->nc2 + RunCfg<2>::SEG - 1) / RunCfg<2>::SEG;
    return mcb_round_up((mcb_round_up(nseg, 128) + RUNS_NTICKETS) * (long long)sizeof(int), 256);
}

bool mcb_runs_supported(const mcb_space* sp) { return sp->M >= 2 && sp->M <= MCB_MAX_M_RUNS && sp->N >= 2; }

long long mcb_runs_workspace_bytes(const mcb_space* sp)
{
    const int NH = sp->M - 2;
    const int ncls = 1 + NH + NH * (NH + 1) / 2;
    return (long long)ncls * runs_ldp(sp) * (long long)sizeof(double2) + runs_sync_bytes(sp);
}

template <int M>
static int launch_runs(mcb_space* sp, const mcb_c128* T, const mcb_c128* V,
                       const mcb_c128* d_C, mcb_c128* d_HC, void* d_ws, cudaStream_t st, const mcb_c128* h_C_src)
{
    using Cfg = RunCfg<M>;
    constexpr int P = Cfg::P;
    // per-space host scratch (a space is used by one thread at a time, include/mcb.h): packed Vp, then the coefficient matrix
    if (!sp->runs_coef) {
        sp->runs_coef = calloc(1, sizeof(RunCoef<M>) + 2 * sizeof(double) * P * P);
        if (!sp->runs_coef) return MCB_ENOMEM;
    }
    RunCoef<M>& coef = *reinterpret_cast<RunCoef<M>*>(sp->runs_coef);
    double* vr = reinterpret_cast<double*>((char*)sp->runs_coef + sizeof(RunCoef<M>));
    double* vi = vr + P * P;
    if (mcb_coef_stale(sp)) {                                            // (held: runs_coef keeps the matrix of the run's first apply)
        mcb_pack_pairs(sp->N, M, T, V, true, vr, vi);
        memset(&coef, 0, sizeof(coef));
        for (int a = 0; a < P; ++a)
            for (int c = 0; c < P; ++c) {
                const double re = vr[a * P + c], im = vi[a * P + c];
                coef.b[2 * c][2 * a] = re;       coef.b[2 * c + 1][2 * a] = -im;
                coef.b[2 * c][2 * a + 1] = im;   coef.b[2 * c + 1][2 * a + 1] = re;
            }
        mcb_coef_staged(sp);
    }

    RunArgs a;
    a.d = sp->dev; a.fock = sp->fock;
    a.C = (const double2*)d_C; a.HC = (double2*)d_HC;
    a.Hp = (double2*)d_ws; a.ldp = runs_ldp(sp);
    a.nseg = (int)((sp->nc2 + Cfg::SEG - 1) / Cfg::SEG);
    a.ntile = (int)((sp->nc + Cfg::SUM_TILE - 1) / Cfg::SUM_TILE);
    {
        const int NH = M - 2;
        const long long planes = (long long)(1 + NH + NH * (NH + 1) / 2) * a.ldp * (long long)sizeof(double2);
        a.tickets = reinterpret_cast<int*>((char*)d_ws + planes);
        a.flags = a.tickets + RUNS_NTICKETS;
    }
    if (!sp->runs_grid) {                                                // cached per space: the space belongs to one device
        int per_sm = 0, sms = 0;
        MCB_CUDA(cudaFuncSetAttribute(k_hc2_runs<M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM));
        MCB_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_hc2_runs<M>, Cfg::THREADS, Cfg::SMEM));
        MCB_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, sp->device));
        if (per_sm < 1) return MCB_EUNSUPPORTED;
        sp->runs_grid = per_sm * sms;
    }
    { int rc = mcb_tick(sp, 0, st); if (rc) return rc; }
    MCB_CUDA(cudaMemsetAsync(a.tickets, 0, (size_t)(mcb_round_up(a.nseg, 128) + RUNS_NTICKETS) * sizeof(int), st));
    ++sp->n_memset;
    a.c_avail = nullptr;
    if (h_C_src) {
        // pipelined host apply: C streams in on the space's copy stream in MCB_H2D_CHUNKS pieces, each followed by a 4-byte
        // copy of the number of elements that have arrived; the kernel starts at once and waits per segment (see next_chunk)
        a.c_avail = a.tickets + 3;
        MCB_CUDA(cudaEventRecord(sp->ev_a, st));
        MCB_CUDA(cudaStreamWaitEvent(sp->copy_stream, sp->ev_a, 0));
        const long long chunk = mcb_round_up((sp->nc + MCB_H2D_CHUNKS - 1) / MCB_H2D_CHUNKS, 4096);
        int i = 0;
        for (long long b = 0; b < sp->nc; b += chunk, ++i) {
            const long long e = b + chunk < sp->nc ? b + chunk : sp->nc;
            MCB_CUDA(cudaMemcpyAsync((mcb_c128*)d_C + b, h_C_src + b, (size_t)(e - b) * sizeof(mcb_c128), cudaMemcpyHostToDevice, sp->copy_stream));
            sp->h_prog[i] = (int)e;
            MCB_CUDA(cudaMemcpyAsync(a.tickets + 3, sp->h_prog + i, sizeof(int), cudaMemcpyHostToDevice, sp->copy_stream));
        }
    }
    k_hc2_runs<M><<<sp->runs_grid, Cfg::THREADS, Cfg::SMEM, st>>>(a, coef);
    MCB_CHECK_LAUNCH();
    if (h_C_src)                                                         // error word of the bounded wait for C -> host (checked after the sync)
        MCB_CUDA(cudaMemcpyAsync(sp->h_prog + MCB_H2D_CHUNKS, a.tickets + 4, sizeof(int), cudaMemcpyDeviceToHost, st));
    { int rc = mcb_tick(sp, 1, st); if (rc) return rc; }
    mcb_tick_done(sp, 1);
    sp->last_launches = 1;
    return MCB_OK;
}

int mcb_launch_runs(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_C, mcb_c128* d_HC,
                    void* d_ws, cudaStream_t st, const mcb_c128* h_C_src)
{
    switch (sp->M) {
    case 2: return launch_runs<2>(sp, T, V, d_C, d_HC, d_ws, st, h_C_src);
    case 3: return launch_runs<3>(sp, T, V, d_C, d_HC, d_ws, st, h_C_src);
    case 4: return launch_runs<4>(sp, T, V, d_C, d_HC, d_ws, st, h_C_src);
    case 5: return launch_runs<5>(sp, T, V, d_C, d_HC, d_ws, st, h_C_src);
    default: return MCB_EUNSUPPORTED;
    }
}
