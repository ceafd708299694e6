// mcb_apply_fma.cu -- MCB_FMA mode of hc_apply (Eq. 12-13) for few orbitals (2 <= M <= 6).
//
// Same factorisation through the (N-2)-particle space as MCB_GEMM (mcb_apply_gemm.cu),
//     H = sum_m sum_{a=(k<=s)} sum_{c=(q<=l)} |m+e_k+e_s> F(m,a) Vp[a][c] F(m,c) <m+e_q+e_l|   (T folded into Vp),
// but laid out for the "few orbitals, many particles" shape (M = 3..5, N = 100..1000), where
// P = M(M+1)/2 is too small to fill DMMA fragments and the index order has long runs:
//
//   * one THREAD per intermediate m.  Its P gathered values D[c] = F(m,c) C[index(m+e_q+e_l)] stay in registers,
//     the packed coefficients Vp arrive as a __grid_constant__ kernel parameter, so every DFMA of the P x P complex
//     mat-vec takes its coefficient straight from the constant bank: no shared memory, no fragment padding, no
//     producer/consumer hand-over.  Consecutive lanes hold consecutive m, so every gather and every store is a
//     contiguous 512-byte warp access along a run.
//   * in-run pre-summation.  Orbitals 0 and 1 only move a configuration inside its run (index +-1), so the
//     removal pairs fall into classes kappa = (the part of e_k+e_s on orbitals >= 2):
//         {}      : (0,0) (0,1) (1,1)          -> outputs g0, g0+1, g0+2 with g0 = index(m + 2 e_0)
//         {h}     : (0,h) (1,h)                -> outputs gh, gh+1       with gh = index(m + e_0 + e_h)
//         {h,h'}  : (h,h')                     -> output  index(m + e_h + e_h')
//     and the contributions of one class to one output come from up to three NEIGHBOURING intermediates of the
//     same run -- neighbouring lanes.  They are summed with warp shuffles and written once into a plane
//     Hp[kappa][g] indexed by the OUTPUT configuration (NCLS = 1 + (M-2) + (M-2)(M-1)/2 planes instead of P),
//     each (kappa, g) slot by exactly one thread: no atomics.
//   * k_hc2_sum<M>: HC[g] = sum over the classes allowed at g of Hp[kappa][g] -- a coalesced stream.
#include <string.h>
#include "mcb_device.cuh"

template <int M> struct FmaCfg {
    static constexpr int P = M * (M + 1) / 2;
    static constexpr int NH = M - 2;                               // orbitals that leave the run
    static constexpr int NCLS = 1 + NH + NH * (NH + 1) / 2;        // classes = planes
    static constexpr int WARPS = 4;
    static constexpr int THREADS = WARPS * 32;
    static constexpr int CHUNKS = 8;                               // 32-wide chunks per warp segment
    static constexpr int SEG = CHUNKS * 32 - 2;                    // intermediates OWNED per segment (2 halo lanes)
    static constexpr int TILE = WARPS * SEG;                       // intermediates per CTA tile
    static constexpr int MINB = (M <= 4) ? 3 : 2;
};

template <int M> struct FmaCoef { double2 v[FmaCfg<M>::P * FmaCfg<M>::P]; };    // Vp[a][c], T folded in

struct FmaArgs {
    McbDev d;
    McbFockView fock;
    const double2* C;
    double2* HC;
    double2* Hp;               // [NCLS][ldp]
    long long ldp;
    int nseg;                  // warp segments
};

__device__ __forceinline__ int fma_cls_single(int h) { return 1 + (h - 2); }
template <int M> __device__ __forceinline__ constexpr int fma_cls_pair(int h, int h2)
{
    // pair index over the NH high orbitals, (h-2) <= (h2-2)
    return 1 + (M - 2) + mcb_pair_index(M - 2, h - 2, h2 - 2);
}

// value of lane (lane - 1), taking lane 31 of the previous chunk for lane 0
__device__ __forceinline__ double2 up1(const double2 cur, const double2 prev, int lane)
{
    const double ax = __shfl_up_sync(0xffffffffu, cur.x, 1), ay = __shfl_up_sync(0xffffffffu, cur.y, 1);
    const double bx = __shfl_sync(0xffffffffu, prev.x, 31), by = __shfl_sync(0xffffffffu, prev.y, 31);
    return lane >= 1 ? make_double2(ax, ay) : make_double2(bx, by);
}
// value of lane (lane - 2), taking lanes 30, 31 of the previous chunk for lanes 0, 1
__device__ __forceinline__ double2 up2(const double2 cur, const double2 prev, int lane)
{
    const double ax = __shfl_up_sync(0xffffffffu, cur.x, 2), ay = __shfl_up_sync(0xffffffffu, cur.y, 2);
    const int src = (lane + 30) & 31;
    const double bx = __shfl_sync(0xffffffffu, prev.x, src), by = __shfl_sync(0xffffffffu, prev.y, src);
    return lane >= 2 ? make_double2(ax, ay) : make_double2(bx, by);
}

// W'[a] = F(m,a) * sum_c Vp[a][c] z[c]; four independent DFMA chains, coefficients from the constant bank
template <int M>
__device__ __forceinline__ double2 fma_row(const FmaCoef<M>& coef, const int a, const double2 (&z)[FmaCfg<M>::P], const double f)
{
    constexpr int P = FmaCfg<M>::P;
    double xr = 0.0, xi = 0.0, yr = 0.0, yi = 0.0;
#pragma unroll
    for (int c = 0; c < P; ++c) {
        const double2 v = coef.v[a * P + c];
        xr = fma(v.x, z[c].x, xr);
        xi = fma(v.y, z[c].y, xi);
        yr = fma(v.x, z[c].y, yr);
        yi = fma(v.y, z[c].x, yi);
    }
    return make_double2(f * (xr - xi), f * (yr + yi));
}

template <int M>
__global__ void __launch_bounds__(FmaCfg<M>::THREADS, FmaCfg<M>::MINB)
k_hc2_contract_fma(const FmaArgs p, const __grid_constant__ FmaCoef<M> coef)
{
    using Cfg = FmaCfg<M>;
    constexpr int P = Cfg::P, NH = Cfg::NH;
    const McbDev& d = p.d;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int seg = blockIdx.x * Cfg::WARPS + warp;
    if (seg >= p.nseg) return;
    const int seg0 = seg * Cfg::SEG;
    const int seg_end = min(seg0 + Cfg::SEG, d.nc2);

    // values of the previous chunk (only lanes 30, 31 are ever consumed)
    double2 prev01 = make_double2(0.0, 0.0), prev11 = make_double2(0.0, 0.0);
    double2 prev1h[NH > 0 ? NH : 1];
#pragma unroll
    for (int h = 0; h < NH; ++h) prev1h[h] = make_double2(0.0, 0.0);

#pragma unroll 1
    for (int ch = 0; ch < Cfg::CHUNKS; ++ch) {
        const int m = seg0 - 2 + ch * 32 + lane;
        if (seg0 - 2 + ch * 32 >= seg_end) break;                       // warp-uniform
        const bool valid = m >= 0 && m < d.nc2;
        const bool own = valid && m >= seg0 && m < seg_end;

        int X[M], Y[M], mj0, mj1;
        double r1[M], r2[M];
        {
            int A1[M], A2[M];
            int run = 0, x = 0, tot1 = 0;
            mj0 = 0; mj1 = 0;
#pragma unroll
            for (int j = 0; j < M; ++j) {
                const int nj = valid ? (int)p.fock.occ2[(long long)j * p.fock.ld2 + m] : 0;
                if (j == 0) mj0 = nj;
                if (j == 1) mj1 = nj;
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
        const int base = d.nc - 1;
        // ---- gather: z[c] = F(m,c) C[index(m + e_q + e_l)] ----
        double2 z[P];
        {
            int c = 0;
#pragma unroll
            for (int q = 0; q < M; ++q) {
#pragma unroll
                for (int l = q; l < M; ++l, ++c)
                    z[c] = valid ? __ldg(p.C + (base - X[q] - Y[l])) : make_double2(0.0, 0.0);
            }
            c = 0;
#pragma unroll
            for (int q = 0; q < M; ++q) {
#pragma unroll
                for (int l = q; l < M; ++l, ++c) {
                    const double f = (q == l) ? r2[q] : r1[q] * r1[l];
                    z[c].x *= f; z[c].y *= f;
                }
            }
        }
        const bool last_in_run = mj0 == 0;
        // ---- class {h,h'}: one pair, one output ----
#pragma unroll
        for (int h = 2; h < M; ++h) {
#pragma unroll
            for (int h2 = h; h2 < M; ++h2) {
                const double f = (h == h2) ? r2[h] : r1[h] * r1[h2];
                const double2 w = fma_row<M>(coef, mcb_pair_index(M, h, h2), z, f);
                if (own) __stcg(p.Hp + (long long)fma_cls_pair<M>(h, h2) * p.ldp + (base - X[h] - Y[h2]), w);
            }
        }
        // ---- class {h}: pairs (0,h), (1,h) ----
#pragma unroll
        for (int h = 2; h < M; ++h) {
            const double2 w0 = fma_row<M>(coef, mcb_pair_index(M, 0, h), z, r1[0] * r1[h]);
            const double2 w1 = fma_row<M>(coef, mcb_pair_index(M, 1, h), z, r1[1] * r1[h]);
            const double2 n1 = up1(w1, prev1h[h - 2], lane);
            prev1h[h - 2] = w1;
            double2 o = w0;
            if (mj1 >= 1) { o.x += n1.x; o.y += n1.y; }
            double2* dst = p.Hp + (long long)fma_cls_single(h) * p.ldp + (base - X[0] - Y[h]);
            if (own) {
                __stcg(dst, o);
                if (last_in_run) __stcg(dst + 1, w1);
            }
        }
        // ---- class {}: pairs (0,0), (0,1), (1,1) ----
        {
            const double2 w00 = fma_row<M>(coef, mcb_pair_index(M, 0, 0), z, r2[0]);
            const double2 w01 = fma_row<M>(coef, mcb_pair_index(M, 0, 1), z, r1[0] * r1[1]);
            const double2 w11 = fma_row<M>(coef, mcb_pair_index(M, 1, 1), z, r2[1]);
            const double2 n01 = up1(w01, prev01, lane);
            const double2 n11a = up1(w11, prev11, lane);
            const double2 n11b = up2(w11, prev11, lane);
            prev01 = w01; prev11 = w11;
            double2 o = w00;
            if (mj1 >= 1) { o.x += n01.x; o.y += n01.y; }
            if (mj1 >= 2) { o.x += n11b.x; o.y += n11b.y; }
            double2* dst = p.Hp + (base - X[0] - Y[0]);
            if (own) {
                __stcg(dst, o);
                if (last_in_run) {
                    double2 e = w01;
                    if (mj1 >= 1) { e.x += n11a.x; e.y += n11a.y; }
                    __stcg(dst + 1, e);
                    __stcg(dst + 2, w11);
                }
            }
        }
    }
}

// HC[g] = sum over the classes allowed at g of Hp[kappa][g]
template <int M>
__global__ void __launch_bounds__(256) k_hc2_sum(const FmaArgs p)
{
    const McbDev& d = p.d;
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= d.nc) return;
    int n[M];
#pragma unroll
    for (int j = 0; j < M; ++j) n[j] = p.fock.occ[(long long)j * p.fock.ld + g];
    const int in01 = n[0] + n[1];
    const double2* src = p.Hp + g;
    double re = 0.0, im = 0.0;
    if (in01 >= 2) { const double2 w = __ldcs(src); re += w.x; im += w.y; }
#pragma unroll
    for (int h = 2; h < M; ++h) {
        if (n[h] >= 1 && in01 >= 1) {
            const double2 w = __ldcs(src + (long long)fma_cls_single(h) * p.ldp);
            re += w.x; im += w.y;
        }
    }
#pragma unroll
    for (int h = 2; h < M; ++h) {
#pragma unroll
        for (int h2 = h; h2 < M; ++h2) {
            const bool ok = (h == h2) ? (n[h] >= 2) : (n[h] >= 1 && n[h2] >= 1);
            if (ok) {
                const double2 w = __ldcs(src + (long long)fma_cls_pair<M>(h, h2) * p.ldp);
                re += w.x; im += w.y;
            }
        }
    }
    p.HC[g] = make_double2(re, im);
}

// =========================================================================================================
// host
// =========================================================================================================
static long long fma_ldp(const mcb_space* sp) { return mcb_round_up(sp->nc, 128); }

bool mcb_fma_supported(const mcb_space* sp) { return sp->M >= 2 && sp->M <= MCB_MAX_M_FMA && sp->N >= 2; }

long long mcb_fma_workspace_bytes(const mcb_space* sp)
{
    const int NH = sp->M - 2;
    const int ncls = 1 + NH + NH * (NH + 1) / 2;
    return (long long)ncls * fma_ldp(sp) * (long long)sizeof(double2);
}

template <int M>
static int launch_fma(mcb_space* sp, const mcb_c128* T, const mcb_c128* V,
                      const mcb_c128* d_C, mcb_c128* d_HC, void* d_ws, cudaStream_t st)
{
    using Cfg = FmaCfg<M>;
    constexpr int P = Cfg::P;
    double* vr = (double*)sp->h_coef;
    double* vi = vr + P * P;
    if ((char*)(vi + P * P) > (char*)sp->h_coef + sp->coef_bytes) return MCB_ENOMEM;
    mcb_pack_pairs(sp->N, M, T, V, true, vr, vi);
    FmaCoef<M> coef;
    for (int i = 0; i < P * P; ++i) coef.v[i] = make_double2(vr[i], vi[i]);

    FmaArgs a;
    a.d = sp->dev; a.fock = sp->fock;
    a.C = (const double2*)d_C; a.HC = (double2*)d_HC;
    a.Hp = (double2*)d_ws; a.ldp = fma_ldp(sp);
    a.nseg = (int)((sp->nc2 + Cfg::SEG - 1) / Cfg::SEG);
    const unsigned grid = (unsigned)((a.nseg + Cfg::WARPS - 1) / Cfg::WARPS);
    { int rc = mcb_tick(sp, 0, st); if (rc) return rc; }
    k_hc2_contract_fma<M><<<grid, Cfg::THREADS, 0, st>>>(a, coef);
    MCB_CHECK_LAUNCH();
    { int rc = mcb_tick(sp, 1, st); if (rc) return rc; }
    const int threads = 256;
    k_hc2_sum<M><<<(unsigned)((sp->nc + threads - 1) / threads), threads, 0, st>>>(a);
    MCB_CHECK_LAUNCH();
    { int rc = mcb_tick(sp, 2, st); if (rc) return rc; }
    mcb_tick_done(sp, 2);
    sp->last_launches = 2;
    return MCB_OK;
}

int mcb_launch_fma(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_C, mcb_c128* d_HC,
                   void* d_ws, cudaStream_t st)
{
    switch (sp->M) {
    case 2: return launch_fma<2>(sp, T, V, d_C, d_HC, d_ws, st);
    case 3: return launch_fma<3>(sp, T, V, d_C, d_HC, d_ws, st);
    case 4: return launch_fma<4>(sp, T, V, d_C, d_HC, d_ws, st);
    case 5: return launch_fma<5>(sp, T, V, d_C, d_HC, d_ws, st);
    case 6: return launch_fma<6>(sp, T, V, d_C, d_HC, d_ws, st);
    default: return MCB_EUNSUPPORTED;
    }
}
