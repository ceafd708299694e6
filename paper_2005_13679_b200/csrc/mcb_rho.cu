// mcb_rho.cu -- one- and two-body density matrices of a coefficient vector (Eq. 10-11; index order
// of App. B):   rho1[k][l] = <Psi|a+_k a_l|Psi>,   rho2[k][s][q][l] = <Psi|a+_k a+_s a_q a_l|Psi>.
//
// Same jump machinery as hc_apply, with the gather-matvec turned into a gather-REDUCTION.
// Through the (N-2)-particle space,  a_q a_l |Psi> = sum_m D_(ql)[m] |m>  with
//     D_c[m] = F(m,c) C[index(m + e_q + e_l)],   F(m,(q,l)) = sqrt((m_q+1)(m_l+1+[q==l])),   c = (q<=l),
// so   rho2[k][s][q][l] = <a_s a_k Psi | a_q a_l Psi> = sum_m conj(D_(ks)[m]) D_(ql)[m] = G[(ks)][(ql)]:
// a P x P complex Gram matrix over nc2 intermediates -- a dense contraction with a very long K, run on the FP64
// tensor path as the real SYRK  S = X X^T,  X = rows (Re D_c, Im D_c) (2P x nc2):
//     Re G[a][c] = S[2a][2c] + S[2a+1][2c+1],   Im G[a][c] = S[2a][2c+1] - S[2a+1][2c].
// rho1 follows from the number operator:  sum_s a+_k a+_s a_s a_l = a+_k N^ a_l = (N-1) a+_k a_l  on N particles.
//
//   k_rho_gram<M>    persistent CTAs walk tiles of TM intermediates: all threads compute the index arithmetic
//                    (mcb_device.cuh), gather C and stage the scaled rows X[r][m] in shared memory; each warp owns a
//                    fixed set of 8 x 8 block pairs (rb <= cb) of S (few pairs, M <= 5: all pairs over its own slice
//                    of the tile) and accumulates them with mma.m8n8k4.f64 (both fragments come from X); at the end
//                    every CTA (warp) writes its partial S once -- no atomics.
//   k_rho_finish     G = sum of the partials, strided + fixed-order tree per element (deterministic).
//   k_rho_expand     rho2 (M^4) and rho1 (M^2) from G; N = 1: rho1 = conj(C_k) C_l, rho2 = 0.
#include <string.h>
#include <mutex>
#include "mcb_device.cuh"

__host__ __device__ constexpr int rho_div(int a, int b) { return (a + b - 1) / b; }

template <int M> struct RhoCfg {
    static constexpr int P = M * (M + 1) / 2;
    static constexpr int RB = rho_div(2 * P, 8);                  // 8-row blocks of X
    static constexpr int ROWS = RB * 8;
    static constexpr int NPAIR = RB * (RB + 1) / 2;               // block pairs rb <= cb of the symmetric S
    static constexpr int WARPS = 8;
    static constexpr int THREADS = WARPS * 32;
    // few block pairs (M <= 5): one thread per intermediate, every warp accumulates ALL pairs over its own 32
    // intermediates of the tile (split K, one partial per warp); otherwise the pairs are dealt out to the warps
    static constexpr bool SPLIT_K = NPAIR <= 16;
    static constexpr int TM = SPLIT_K ? THREADS : 64;             // intermediates per tile
    static constexpr int LD = TM + 4;                             // row stride in doubles (LD % 16 == 4: conflict-free fragments)
    static constexpr int NPART = THREADS / TM;                    // threads per intermediate in the gather
    static constexpr int PPW = SPLIT_K ? NPAIR : rho_div(NPAIR, WARPS);   // block pairs per warp
    static constexpr int KS0 = SPLIT_K ? 8 : 0;                   // k-steps (of 4 intermediates) per warp slice
    static constexpr int NKS = SPLIT_K ? 8 : TM / 4;
    static constexpr size_t SMEM = (size_t)ROWS * LD * sizeof(double);
};

struct RhoArgs {
    McbDev d;
    McbFockView fock;
    const double2* C;
    double* partial;           // [gridDim][ROWS][ROWS], only blocks rb <= cb are written
    int ntiles;
};

__device__ __forceinline__ void rho_dmma884(double& c0, double& c1, const double a, const double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <int M>
__global__ void __launch_bounds__(RhoCfg<M>::THREADS) k_rho_gram(const RhoArgs p)
{
    using Cfg = RhoCfg<M>;
    constexpr int RB = Cfg::RB, TM = Cfg::TM, LD = Cfg::LD;
    extern __shared__ double rho_X[];                                    // [ROWS][LD]
    const McbDev& d = p.d;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int grp = lane >> 2, tig = lane & 3;
    for (int i = tid; i < Cfg::ROWS * LD; i += Cfg::THREADS) rho_X[i] = 0.0;        // padding rows stay zero

    // the block pairs this warp owns: pair index -> (rb, cb), rb <= cb, order (0,0),(0,1),..,(0,RB-1),(1,1),..
    int prb[Cfg::PPW], pcb[Cfg::PPW];
    double acc[Cfg::PPW][2];
#pragma unroll
    for (int i = 0; i < Cfg::PPW; ++i) {
        int q = Cfg::SPLIT_K ? i : warp + i * Cfg::WARPS, rb = 0, len = RB;
        if (q >= Cfg::NPAIR) { prb[i] = -1; pcb[i] = 0; }
        else { while (q >= len) { q -= len; --len; ++rb; } prb[i] = rb; pcb[i] = rb + q; }
        acc[i][0] = 0.0; acc[i][1] = 0.0;
    }
    const int ml = tid % TM, part = tid / TM;
    __syncthreads();

    for (int tile = blockIdx.x; tile < p.ntiles; tile += gridDim.x) {
        // ---- gather: X[2c][ml] + i X[2c+1][ml] = F(m,c) C[index(m + e_q + e_l)] ----
        {
            const int m = tile * TM + ml;
            const bool valid = m < d.nc2;
            int X[M], Y[M];
            double r1[M], r2[M];
            {
                int A1[M], A2[M];
                int run = 0, x = 0, tot1 = 0;
#pragma unroll
                for (int j = 0; j < M; ++j) {
                    const int nj = valid ? (int)p.fock.occ2[(long long)j * p.fock.ld2 + m] : 0;
                    run += nj;
                    r1[j] = __ldg(d.sq + nj + 1);
                    r2[j] = __ldg(d.sq2 + nj + 2);
                    X[j] = x;
                    if (j <= M - 2) {
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
            int c = 0;
#pragma unroll
            for (int q = 0; q < M; ++q) {
#pragma unroll
                for (int l = q; l < M; ++l, ++c) {
                    if (c % Cfg::NPART == part) {
                        const double2 z = valid ? __ldg(p.C + MCB_CHK(d, d.nc - 1 - X[q] - Y[l], d.nc, 701)) : make_double2(0.0, 0.0);
                        const double f = (q == l) ? r2[q] : r1[q] * r1[l];
                        rho_X[(2 * c) * LD + ml] = f * z.x;
                        rho_X[(2 * c + 1) * LD + ml] = f * z.y;
                    }
                }
            }
        }
        __syncthreads();
        // ---- S[rb][cb] += X_rb X_cb^T over the TM intermediates of the tile ----
#pragma unroll
        for (int i = 0; i < Cfg::PPW; ++i) {
            if (prb[i] < 0) continue;                                    // warp-uniform
            const double* xa = rho_X + (prb[i] * 8 + grp) * LD + tig + warp * Cfg::KS0 * 4;
            const double* xb = rho_X + (pcb[i] * 8 + grp) * LD + tig + warp * Cfg::KS0 * 4;
#pragma unroll
            for (int ks = 0; ks < Cfg::NKS; ++ks) rho_dmma884(acc[i][0], acc[i][1], xa[ks * 4], xb[ks * 4]);
        }
        __syncthreads();
    }
    double* out = p.partial + (size_t)(Cfg::SPLIT_K ? blockIdx.x * Cfg::WARPS + warp : blockIdx.x) * Cfg::ROWS * Cfg::ROWS;
#pragma unroll
    for (int i = 0; i < Cfg::PPW; ++i) {
        if (prb[i] < 0) continue;
        double* o = out + (size_t)(prb[i] * 8 + grp) * Cfg::ROWS + pcb[i] * 8 + 2 * tig;
        o[0] = acc[i][0];
        o[1] = acc[i][1];
    }
}

// G[a][c] = sum over CTAs of (S[2a][2c] + S[2a+1][2c+1]) + i (S[2a][2c+1] - S[2a+1][2c]); S(i,j) is stored for
// block(i) <= block(j) only.
__global__ void __launch_bounds__(128) k_rho_finish(const double* __restrict__ partial, int nblocks, int ROWS, int P, double2* __restrict__ G)
{
    // one CTA per element (a, c): threads stride over the partials, then a fixed-order tree reduction
    __shared__ double sre[128], sim[128];
    const int e = blockIdx.x;
    const int a = e / P, c = e % P;
    auto at = [&](const double* S, int i, int j) { return (i >> 3) <= (j >> 3) ? S[(size_t)i * ROWS + j] : S[(size_t)j * ROWS + i]; };
    double re = 0.0, im = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += 128) {
        const double* S = partial + (size_t)b * ROWS * ROWS;
        re += at(S, 2 * a, 2 * c) + at(S, 2 * a + 1, 2 * c + 1);
        im += at(S, 2 * a, 2 * c + 1) - at(S, 2 * a + 1, 2 * c);
    }
    sre[threadIdx.x] = re; sim[threadIdx.x] = im;
    __syncthreads();
    for (int w = 64; w >= 1; w >>= 1) {
        if (threadIdx.x < w) { sre[threadIdx.x] += sre[threadIdx.x + w]; sim[threadIdx.x] += sim[threadIdx.x + w]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) G[e] = make_double2(sre[0], sim[0]);
}

__global__ void k_rho_expand(const double2* __restrict__ G, const double2* __restrict__ C, int N, int M,
                             double2* __restrict__ rho1, double2* __restrict__ rho2)
{
    const int M2 = M * M;
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < M2 * M2) {
        const int k = e / (M2 * M), s = (e / M2) % M, q = (e / M) % M, l = e % M;
        double2 v = make_double2(0.0, 0.0);
        if (N >= 2) {
            const int P = M * (M + 1) / 2;
            const int a = mcb_pair_index(M, min(k, s), max(k, s)), c = mcb_pair_index(M, min(q, l), max(q, l));
            v = G[a * P + c];
        }
        rho2[e] = v;
    }
    if (e < M2) {
        const int k = e / M, l = e % M;
        double2 v = make_double2(0.0, 0.0);
        if (N >= 2) {
            const int P = M * (M + 1) / 2;
            for (int s = 0; s < M; ++s) {
                const double2 g = G[mcb_pair_index(M, min(k, s), max(k, s)) * P + mcb_pair_index(M, min(s, l), max(s, l))];
                v.x += g.x; v.y += g.y;
            }
            v.x /= (double)(N - 1); v.y /= (double)(N - 1);
        } else {                                                         // N = 1: Algorithm 1 gives |e_j> the index N_c(1, j) = j
            const double2 ck = C[k], cl = C[l];
            v = make_double2(ck.x * cl.x + ck.y * cl.y, ck.x * cl.y - ck.y * cl.x);
        }
        rho1[e] = v;
    }
}

// =========================================================================================================
// host
// =========================================================================================================
static int rho_grid(const mcb_space* sp)
{
    // persistent CTAs per SM the kernel is shaped for (registers / shared memory): 4 for M <= 5, 2 up to M = 8, else 1
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, sp->device) != cudaSuccess || sms < 1) sms = 148;
    return (sp->M <= 5 ? 4 : (sp->M <= 8 ? 2 : 1)) * sms;
}
static int rho_rows(int M) { const int P = M * (M + 1) / 2; return (2 * P + 7) / 8 * 8; }
// partial matrices per CTA: one per warp when K is split (RhoCfg::SPLIT_K: at most 16 block pairs)
static int rho_parts(int M) { const int rb = rho_rows(M) / 8; return rb * (rb + 1) / 2 <= 16 ? 8 : 1; }

int mcb_rho_expand_launch(const void* d_G, const mcb_c128* d_C, int N, int M, mcb_c128* d_rho1, mcb_c128* d_rho2, cudaStream_t st)
{
    const int M4 = M * M * M * M;
    k_rho_expand<<<(M4 + 127) / 128, 128, 0, st>>>((const double2*)d_G, (const double2*)d_C, N, M, (double2*)d_rho1, (double2*)d_rho2);
    MCB_CHECK_LAUNCH();
    return MCB_OK;
}

extern "C" long long mcb_rho_workspace_bytes(const mcb_space* sp)
{
    if (!sp) return MCB_EINVAL;
    if (sp->M > MCB_MAX_M_APPLY) return MCB_EUNSUPPORTED;
    if (sp->M > MCB_MAX_M_TILED) return mcb_big_rho_workspace_bytes(sp);
    const long long rows = rho_rows(sp->M);
    const long long partial = mcb_round_up((long long)rho_grid(sp) * rho_parts(sp->M) * rows * rows * (long long)sizeof(double), 256);
    return partial + mcb_round_up((long long)sp->P * sp->P * (long long)sizeof(double2), 256);
}

template <int M>
static int launch_rho(mcb_space* sp, const mcb_c128* d_C, mcb_c128* d_rho1, mcb_c128* d_rho2, void* d_ws, cudaStream_t st)
{
    using Cfg = RhoCfg<M>;
    const int grid_max = rho_grid(sp);
    static_assert(Cfg::WARPS == 8, "rho_parts");
    const long long partial_bytes = mcb_round_up((long long)grid_max * rho_parts(M) * Cfg::ROWS * Cfg::ROWS * (long long)sizeof(double), 256);
    double* partial = (double*)d_ws;
    double2* G = (double2*)((char*)d_ws + partial_bytes);
    int launches = 0;
    if (sp->N >= 2) {
        RhoArgs a;
        a.d = sp->dev; a.fock = sp->fock; a.C = (const double2*)d_C; a.partial = partial;
        a.ntiles = (int)((sp->nc2 + Cfg::TM - 1) / Cfg::TM);
        const int grid = a.ntiles < grid_max ? a.ntiles : grid_max;
        if (!(sp->attr_set & 1u)) {                                      // per space: the attribute is per device
            MCB_CUDA(cudaFuncSetAttribute(k_rho_gram<M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM));
            sp->attr_set |= 1u;
        }
        k_rho_gram<M><<<grid, Cfg::THREADS, Cfg::SMEM, st>>>(a);
        MCB_CHECK_LAUNCH();
        k_rho_finish<<<Cfg::P * Cfg::P, 128, 0, st>>>(partial, grid * rho_parts(M), Cfg::ROWS, Cfg::P, G);
        MCB_CHECK_LAUNCH();
        launches = 2;
    }
    const int M4 = M * M * M * M;
    k_rho_expand<<<(M4 + 127) / 128, 128, 0, st>>>(G, (const double2*)d_C, sp->N, M, (double2*)d_rho1, (double2*)d_rho2);
    MCB_CHECK_LAUNCH();
    sp->last_launches = launches + 1;
    return MCB_OK;
}

extern "C" int mcb_rho(mcb_space* sp, const mcb_c128* d_C, mcb_c128* d_rho1, mcb_c128* d_rho2, void* d_workspace, void* stream)
{
    if (!sp || !d_C || !d_rho1 || !d_rho2 || !d_workspace) return MCB_EINVAL;
    if (sp->M > MCB_MAX_M_APPLY) return MCB_EUNSUPPORTED;
    if ((((uintptr_t)d_C) & 15) || (((uintptr_t)d_rho1) & 15) || (((uintptr_t)d_rho2) & 15) || (((uintptr_t)d_workspace) & 255))
        return MCB_EINVAL;
    if (sp->N >= 2 && !sp->d_fock) return MCB_ENOTREADY;
    cudaStream_t st = (cudaStream_t)stream;
    if (sp->M > MCB_MAX_M_TILED) return mcb_launch_rho_big(sp, d_C, d_rho1, d_rho2, d_workspace, st);
    switch (sp->M) {
    case 1: return launch_rho<1>(sp, d_C, d_rho1, d_rho2, d_workspace, st);
    case 2: return launch_rho<2>(sp, d_C, d_rho1, d_rho2, d_workspace, st);
    case 3: return launch_rho<3>(sp, d_C, d_rho1, d_rho2, d_workspace, st);
    case 4: return launch_rho<4>(sp, d_C, d_rho1, d_rho2, d_workspace, st);
    case 5: return launch_rho<5>(sp, d_C, d_rho1, d_rho2, d_workspace, st);
    case 6: return launch_rho<6>(sp, d_C, d_rho1, d_rho2, d_workspace, st);
    case 7: return launch_rho<7>(sp, d_C, d_rho1, d_rho2, d_workspace, st);
    case 8: return launch_rho<8>(sp, d_C, d_rho1, d_rho2, d_workspace, st);
    case 9: return launch_rho<9>(sp, d_C, d_rho1, d_rho2, d_workspace, st);
    case 10: return launch_rho<10>(sp, d_C, d_rho1, d_rho2, d_workspace, st);
    case 11: return launch_rho<11>(sp, d_C, d_rho1, d_rho2, d_workspace, st);
    case 12: return launch_rho<12>(sp, d_C, d_rho1, d_rho2, d_workspace, st);
    default: return MCB_EUNSUPPORTED;
    }
}

// =========================================================================================================
// mcb_rho_static: the same three kernels with their scratch in a fixed array of this library (include/mcb.h)
// =========================================================================================================
// Who this is for: code that is handed its device buffers by a host program and has no way to ask for more -- a solver plugged
// into an application whose own pool took the whole device at start-up (a cudaMalloc there fails, or breaks the memory budget
// the job was given), or a propagation loop in which cudaMalloc / cudaFree are forbidden because they synchronise the whole
// device and hold a driver lock that stalls every other stream and thread of the process.  Such a caller owns C and the two
// result matrices but cannot produce the mcb_rho_workspace_bytes() of scratch mcb_rho wants.  Here the partial Gram matrices
// of k_rho_gram and the reduced G of k_rho_finish live in MCB_RHO_STATIC_BYTES of device memory that belongs to the library
// image: every device that loads libmcb.so carries it from the first use of this file's kernels until the process exits.
//
// In HOST code `rho_static_scratch` is only a handle of the symbol (using it as a pointer would hand the kernels a host
// address); the device address differs per device and comes from cudaGetSymbolAddress with that device current, looked up
// the first time this entry point runs on a device and remembered per device ordinal.
static __device__ __align__(256) unsigned char rho_static_scratch[MCB_RHO_STATIC_BYTES];

#define RHO_STATIC_MAX_DEVICES 64
static std::mutex rho_static_mutex;
static void* rho_static_ptr[RHO_STATIC_MAX_DEVICES];                     // device address of rho_static_scratch, by device ordinal

static int rho_static_address(int device, void** out)
{
    std::lock_guard<std::mutex> lock(rho_static_mutex);
    void* p = (device >= 0 && device < RHO_STATIC_MAX_DEVICES) ? rho_static_ptr[device] : NULL;
    if (!p) {                                                            // (the caller has checked that `device` is current)
        MCB_CUDA(cudaGetSymbolAddress(&p, rho_static_scratch));
        if (!p || (((uintptr_t)p) & 255)) return MCB_ECUDA;
        if (device >= 0 && device < RHO_STATIC_MAX_DEVICES) rho_static_ptr[device] = p;
    }
    *out = p;
    return MCB_OK;
}

template <int M>
static int launch_rho_static(mcb_space* sp, const mcb_c128* d_C, mcb_c128* d_rho1, mcb_c128* d_rho2, void* scratch, cudaStream_t st)
{
    using Cfg = RhoCfg<M>;
    // scratch layout: G [P][P] complex | per-CTA partial matrices.  The persistent grid is cut to the number of partials the
    // array holds (k_rho_gram strides over the tiles by gridDim.x, so any grid >= 1 is a correct one).
    const long long g_bytes = mcb_round_up((long long)Cfg::P * Cfg::P * (long long)sizeof(double2), 256);
    const long long per_cta = (long long)rho_parts(M) * Cfg::ROWS * Cfg::ROWS * (long long)sizeof(double);
    const long long grid_cap = ((long long)MCB_RHO_STATIC_BYTES - g_bytes) / per_cta;
    if (grid_cap < 1) return MCB_ESCRATCH;
    double2* G = (double2*)scratch;
    double* partial = (double*)((char*)scratch + g_bytes);
    int launches = 0;
    if (sp->N >= 2) {
        RhoArgs a;
        a.d = sp->dev; a.fock = sp->fock; a.C = (const double2*)d_C; a.partial = partial;
        a.ntiles = (int)((sp->nc2 + Cfg::TM - 1) / Cfg::TM);
        long long grid = rho_grid(sp);
        if (grid > a.ntiles) grid = a.ntiles;
        if (grid > grid_cap) grid = grid_cap;
        if (!(sp->attr_set & 1u)) {
            MCB_CUDA(cudaFuncSetAttribute(k_rho_gram<M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM));
            sp->attr_set |= 1u;
        }
        // nothing in the array has to start at zero: every CTA (warp) of this grid stores all of its block pairs, and
        // k_rho_finish reads exactly grid * rho_parts partials -- what an earlier call left behind is never looked at
        k_rho_gram<M><<<(int)grid, Cfg::THREADS, Cfg::SMEM, st>>>(a);
        MCB_CHECK_LAUNCH();
        k_rho_finish<<<Cfg::P * Cfg::P, 128, 0, st>>>(partial, (int)grid * rho_parts(M), Cfg::ROWS, Cfg::P, G);
        MCB_CHECK_LAUNCH();
        launches = 2;
    }
    const int M4 = M * M * M * M;
    k_rho_expand<<<(M4 + 127) / 128, 128, 0, st>>>(G, (const double2*)d_C, sp->N, M, (double2*)d_rho1, (double2*)d_rho2);
    MCB_CHECK_LAUNCH();
    sp->last_launches = launches + 1;
    return MCB_OK;
}

extern "C" int mcb_rho_static(mcb_space* sp, const mcb_c128* d_C, mcb_c128* d_rho1, mcb_c128* d_rho2, void* stream)
{
    if (!sp || !d_C || !d_rho1 || !d_rho2) return MCB_EINVAL;
    if ((((uintptr_t)d_C) & 15) || (((uintptr_t)d_rho1) & 15) || (((uintptr_t)d_rho2) & 15)) return MCB_EINVAL;
    if (sp->M > MCB_RHO_STATIC_MAX_M) return MCB_ESCRATCH;               // beyond: P x nc2 materialised rows, no fixed bound
    if (sp->N >= 2 && !sp->d_fock) return MCB_ENOTREADY;
    int device = -1;
    MCB_CUDA(cudaGetDevice(&device));
    if (device != sp->device) return MCB_EINVAL;                         // the space's tables live on the device it was created on
    void* scratch = NULL;
    const int rc = rho_static_address(device, &scratch);
    if (rc != MCB_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    switch (sp->M) {
    case 1: return launch_rho_static<1>(sp, d_C, d_rho1, d_rho2, scratch, st);
    case 2: return launch_rho_static<2>(sp, d_C, d_rho1, d_rho2, scratch, st);
    case 3: return launch_rho_static<3>(sp, d_C, d_rho1, d_rho2, scratch, st);
    case 4: return launch_rho_static<4>(sp, d_C, d_rho1, d_rho2, scratch, st);
    case 5: return launch_rho_static<5>(sp, d_C, d_rho1, d_rho2, scratch, st);
    case 6: return launch_rho_static<6>(sp, d_C, d_rho1, d_rho2, scratch, st);
    case 7: return launch_rho_static<7>(sp, d_C, d_rho1, d_rho2, scratch, st);
    case 8: return launch_rho_static<8>(sp, d_C, d_rho1, d_rho2, scratch, st);
    case 9: return launch_rho_static<9>(sp, d_C, d_rho1, d_rho2, scratch, st);
    case 10: return launch_rho_static<10>(sp, d_C, d_rho1, d_rho2, scratch, st);
    case 11: return launch_rho_static<11>(sp, d_C, d_rho1, d_rho2, scratch, st);
    case 12: return launch_rho_static<12>(sp, d_C, d_rho1, d_rho2, scratch, st);
    default: return MCB_ESCRATCH;
    }
}
