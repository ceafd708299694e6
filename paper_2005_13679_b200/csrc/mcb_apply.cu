// mcb_apply.cu -- HC = H.C (Eq. 12-13) on one B200.
//
// Three device paths (include/mcb.h "hc_apply modes"):
//   k_hc_direct<M, false>  MCB_REHASH: one thread per output configuration g, every target index recomputed
//                          on the fly from the hashing table ("hashing table + algorithm 1",
//                          with Algorithm 1 collapsed to O(M) look-ups);
//   k_hc_direct<M, true>   MCB_MAPS:   same loop nest, target indices streamed from Map1 / Map2;
//   k_hc2_contract<M> + k_hc2_reduce<M>   MCB_GEMM: the two-body operator factored through the (N-2)-particle
//                          space,  H2 = sum_m sum_{(k<=s),(q<=l)} |m+e_k+e_s> F(m,ks) Vp[ks][ql] F(m,ql) <m+e_q+e_l|,
//                          F(m,ql) = sqrt((m_q+1)(m_l+1+[q==l])), so that per intermediate m the work is a dense
//                          P x P complex mat-vec -- batched over m: an FP64 tensor-core (DMMA) GEMM with the
//                          packed V stationary in registers.  T rides along inside V (sum_s a+_s a_s = N).
#include <stdlib.h>
#include <string.h>
#include "mcb_device.cuh"

// =========================================================================================================
// host: packing of T, V
// =========================================================================================================

// Vp[a][c], a = pair(k<=s), c = pair(q<=l):  1/2 * sum over the DISTINCT orderings (k',s') of {k,s} and (q',l')
// of {q,l} of Veff[k'][s'][q'][l'].  The bosonic operator a+_k a+_s a_q a_l is symmetric under k<->s and q<->l,
// so the ordered sum of Eq. (13) equals the sum over unordered pairs of Vp times the operator (reading A8).
// With fold_T, Veff = V + (2/(N-1)) T[k][l] delta_sq, which adds sum_kl T_kl a+_k (N^ ) a_l / (N-1) = the one-body
// term on N-particle states.
void mcb_pack_pairs(int N, int M, const mcb_c128* T, const mcb_c128* V, bool fold_T, double* vr, double* vi /* [P][P] */)
{
    const int P = M * (M + 1) / 2;
    const double tf = (fold_T && N >= 2) ? 2.0 / (double)(N - 1) : 0.0;
    int a = 0;
    for (int k = 0; k < M; ++k)
        for (int s = k; s < M; ++s, ++a) {
            int c = 0;
            for (int q = 0; q < M; ++q)
                for (int l = q; l < M; ++l, ++c) {
                    double re = 0.0, im = 0.0;
                    const int nks = (k == s) ? 1 : 2, nql = (q == l) ? 1 : 2;
                    for (int i = 0; i < nks; ++i)
                        for (int j = 0; j < nql; ++j) {
                            const int kk = i ? s : k, ss = i ? k : s, qq = j ? l : q, ll = j ? q : l;
                            const mcb_c128 v = V[(((size_t)kk * M + ss) * M + qq) * M + ll];
                            re += v.re; im += v.im;
                            if (tf != 0.0 && ss == qq) {
                                const mcb_c128 t = T[(size_t)kk * M + ll];
                                re += tf * t.re; im += tf * t.im;
                            }
                        }
                    vr[(size_t)a * P + c] = 0.5 * re;
                    vi[(size_t)a * P + c] = 0.5 * im;
                }
        }
}

// =========================================================================================================
// direct per-output kernel (MCB_REHASH / MCB_MAPS)
// =========================================================================================================
struct DirectArgs {
    McbDev d;
    McbFockView fock;
    const double2* C;
    double2* HC;
    const double2* coef;       // [M*M] T, then [P*P] Vp (ks-major)
    const int* map1; long long ld1;
    const int* map2; long long ld2;
};

__device__ __forceinline__ void cfma(double2& acc, const double2 a, const double2 b)
{
    acc.x = fma(a.x, b.x, acc.x); acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y); acc.y = fma(a.y, b.x, acc.y);
}

// a map entry is read exactly once per apply: keep the stream out of L1, which the gathers of C need
#ifndef MAPLD
#define MAPLD 1
#endif
__device__ __forceinline__ int ld_map(const int* ptr)
{
#if MAPLD == 1
    int v;
    asm("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(v) : "l"(ptr));
    return v;
#elif MAPLD == 2
    return __ldcs(ptr);
#else
    return __ldg(ptr);
#endif
}

template <int M, bool USE_MAPS>
__global__ void __launch_bounds__(128) k_hc_direct(DirectArgs p)
{
    constexpr int P = M * (M + 1) / 2;
    extern __shared__ double2 s_coef[];                     // T [M*M], Vp [P*P]
    for (int i = threadIdx.x; i < M * M + P * P; i += blockDim.x) s_coef[i] = p.coef[i];
    __syncthreads();
    const double2* sT = s_coef;
    const double2* sV = s_coef + M * M;
    const McbDev& d = p.d;
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= d.nc) return;

    int n[M], S[M];
    {
        int run = 0;
#pragma unroll
        for (int j = 0; j < M; ++j) { n[j] = p.fock.occ[(long long)j * p.fock.ld + g]; run += n[j]; S[j] = run; }
    }
    double2 acc = make_double2(0.0, 0.0);
    const double2 cg = p.C[g];
    // on-the-fly rehashing, few pairs: every prefix sum the index arithmetic can meet is S_j + delta, delta in -2..2, so
    // the table entries G[j][S_j - 2 .. S_j + 2] are fetched once per output (5 (M-1) look-ups instead of 9 (M-1) per
    // allowed removal pair); with the pair loops unrolled every use is a compile-time register pick
    constexpr bool CACHE = !USE_MAPS && P <= 15;
    int GG[CACHE ? (M > 1 ? M - 1 : 1) : 1][5];
    if (CACHE) {
#pragma unroll
        for (int j = 0; j + 1 < M; ++j)
#pragma unroll
            for (int t = 0; t < 5; ++t) GG[j][t] = mcb_ldG(d.G, d.ldg, j, min(max(S[j] + t - 2, 0), d.N));
    }

    // ---- one-body: sum_kl T_kl sqrt(n_k (n_l + 1)) C[g_k^l], diagonal n_k C[g]  (App. B rho_kl, rho_kk) ----
    {
        int PM[M], PP[M];
        if (!USE_MAPS) {
            int pm = 0, pp = 0;
#pragma unroll
            for (int j = 0; j < M; ++j) {
                PM[j] = pm; PP[j] = pp;
                if (j <= M - 2) {
                    int g0 = CACHE ? GG[j][2] : mcb_ldG(d.G, d.ldg, j, S[j]);
                    int gm = CACHE ? GG[j][1] : mcb_ldG(d.G, d.ldg, j, S[j] > 0 ? S[j] - 1 : 0);
                    int gp = CACHE ? GG[j][3] : mcb_ldG(d.G, d.ldg, j, S[j] < d.N ? S[j] + 1 : d.N);
                    pm += g0 - gm; pp += gp - g0;
                }
            }
        }
        double rk[M], rl[M];
#pragma unroll
        for (int j = 0; j < M; ++j) { rk[j] = __ldg(d.sq + n[j]); rl[j] = __ldg(d.sq + n[j] + 1); }
#pragma unroll
        for (int k = 0; k < M; ++k) {
            if (n[k] >= 1) {
#pragma unroll
                for (int l = 0; l < M; ++l) {
                    const double2 t = sT[k * M + l];
                    if (l == k) {
                        const double f = (double)n[k];
                        cfma(acc, t, make_double2(f * cg.x, f * cg.y));
                    } else {
                        int tgt;
                        if (USE_MAPS) tgt = ld_map(p.map1 + (long long)(k * M + l) * p.ld1 + g);
                        else tgt = (k < l) ? g + (PM[l] - PM[k]) : g - (PP[k] - PP[l]);
                        const double2 c = __ldg(p.C + MCB_CHK(d, tgt, d.nc, 101));
                        const double f = rk[k] * rl[l];
                        cfma(acc, t, make_double2(f * c.x, f * c.y));
                    }
                }
            }
        }
    }

    // ---- two-body: sum over allowed removal pairs (k<=s), then all insertion pairs (q<=l) ----
    if (d.N >= 2) {
        constexpr int PAIR_UNROLL = CACHE ? M : 1;
        constexpr bool MAP_PREFETCH = USE_MAPS && P <= 15;               // two target buffers in registers
        int tcur[MAP_PREFETCH ? P : 1], tnext[MAP_PREFETCH ? P : 1];
        if (MAP_PREFETCH) {
#pragma unroll
            for (int cc = 0; cc < P; ++cc) tnext[MAP_PREFETCH ? cc : 0] = ld_map(p.map2 + (long long)cc * p.ld2 + g);
        }
        int a_run = 0;                                                   // pair counter of the rolled loops
#pragma unroll PAIR_UNROLL
        for (int k = 0; k < M; ++k) {
#pragma unroll PAIR_UNROLL
            for (int s = CACHE ? 0 : k; s < M; ++s, a_run += CACHE ? 0 : 1) {
                if (CACHE && s < k) continue;                            // (full trip count so that the loop unrolls)
                const int a = CACHE ? mcb_pair_index(M, k, s) : a_run;
                int nk = 0, ns = 0;
#pragma unroll
                for (int j = 0; j < M; ++j) { nk = (j == k) ? n[j] : nk; ns = (j == s) ? n[j] : ns; }
                const bool ok = (k == s) ? (nk >= 2) : (nk >= 1 && ns >= 1);
                if (MAP_PREFETCH) {
                    // the targets of this pair were loaded one pair ago; those of the next pair (whether it is allowed or not: the
                    // planes of forbidden removals hold -1) are loaded before this pair's gathers are issued (a second pair of
                    // look-ahead changes nothing: 1.75 against 1.71 ms at configs[2])
#pragma unroll
                    for (int cc = 0; cc < P; ++cc) tcur[cc] = tnext[cc];
                    if (a + 1 < P) {
                        const int* m2n = p.map2 + (long long)(a + 1) * P * p.ld2 + g;
#pragma unroll
                        for (int cc = 0; cc < P; ++cc) tnext[cc] = ld_map(m2n + (long long)cc * p.ld2);
                    }
                }
                if (!ok) continue;
                const double f1 = (k == s) ? __ldg(d.sq2 + nk) : __ldg(d.sq + nk) * __ldg(d.sq + ns);
                double r1[M], r2[M];
                int X[M], Y[M];
                {
                    int A1[M], A2[M];
                    int x = 0, tot1 = 0;
#pragma unroll
                    for (int j = 0; j < M; ++j) {
                        const int mj = n[j] - (j == k) - (j == s);
                        r1[j] = __ldg(d.sq + mj + 1);
                        r2[j] = __ldg(d.sq2 + mj + 2);
                        X[j] = x;
                        if (!USE_MAPS && j <= M - 2) {
                            const int sp = S[j] - (j >= k) - (j >= s);
                            const int dlt = 2 - (j >= k) - (j >= s);             // compile time when the pair loops are unrolled
                            const int a0 = CACHE ? GG[j][dlt] : mcb_ldG(d.G, d.ldg, j, sp);
                            A1[j] = CACHE ? GG[j][dlt + 1] : mcb_ldG(d.G, d.ldg, j, sp + 1);
                            A2[j] = CACHE ? GG[j][dlt + 2] : mcb_ldG(d.G, d.ldg, j, sp + 2);
                            x += a0 - A1[j]; tot1 += A1[j];
                        } else { A1[j] = 0; A2[j] = 0; }
                    }
                    int pre = tot1, suf = 0;
#pragma unroll
                    for (int l = M - 1; l >= 0; --l) { pre -= A1[l]; suf += A2[l]; Y[l] = pre + suf; }
                }
                double2 w = make_double2(0.0, 0.0);
                const double2* vrow = sV + a * P;
                const int* m2 = USE_MAPS ? p.map2 + (long long)a * P * p.ld2 + g : nullptr;
                int c = 0;
#pragma unroll
                for (int q = 0; q < M; ++q) {
#pragma unroll
                    for (int l = q; l < M; ++l, ++c) {
                        const int tgt = MAP_PREFETCH ? tcur[c] : (USE_MAPS ? ld_map(m2 + (long long)c * p.ld2) : d.nc - 1 - X[q] - Y[l]);
                        const double2 z = __ldg(p.C + MCB_CHK(d, tgt, d.nc, 102));
                        const double f2 = (q == l) ? r2[q] : r1[q] * r1[l];
                        cfma(w, vrow[c], make_double2(f2 * z.x, f2 * z.y));
                    }
                }
                acc.x = fma(f1, w.x, acc.x);
                acc.y = fma(f1, w.y, acc.y);
            }
        }
    }
    p.HC[g] = acc;
}

// =========================================================================================================
// host entry points
// =========================================================================================================
#define MCB_DISPATCH_APPLY_M(M, CALL)                                                                    \
    switch (M) {                                                                                         \
    case 1:  { constexpr int MT = 1;  CALL; } break;  case 2:  { constexpr int MT = 2;  CALL; } break;   \
    case 3:  { constexpr int MT = 3;  CALL; } break;  case 4:  { constexpr int MT = 4;  CALL; } break;   \
    case 5:  { constexpr int MT = 5;  CALL; } break;  case 6:  { constexpr int MT = 6;  CALL; } break;   \
    case 7:  { constexpr int MT = 7;  CALL; } break;  case 8:  { constexpr int MT = 8;  CALL; } break;   \
    case 9:  { constexpr int MT = 9;  CALL; } break;  case 10: { constexpr int MT = 10; CALL; } break;   \
    case 11: { constexpr int MT = 11; CALL; } break;  case 12: { constexpr int MT = 12; CALL; } break;   \
    default: return MCB_EUNSUPPORTED;                                                                    \
    }

static int resolve_mode(const mcb_space* sp, int mode)
{
    // the persistent MCB_RUNS kernel (tickets, flags, a memset) pays off from about a million configurations on
    // (measured: N = 1000, M = 3, nc = 5.0e5: 52 us against 36 us for MCB_GEMM; N = 2000, nc = 2.0e6: 96 against 128 us)
    if (mode == MCB_AUTO)
        return sp->N < 2 ? MCB_REHASH : ((mcb_runs_supported(sp) && sp->nc >= (1LL << 20)) ? MCB_RUNS : MCB_GEMM);
    if ((mode == MCB_GEMM || mode == MCB_RUNS) && sp->N < 2) return MCB_REHASH;   // no (N-2)-particle space: one-body only
    return mode;
}

extern "C" long long mcb_apply_workspace_bytes(const mcb_space* sp, int mode)
{
    if (!sp) return MCB_EINVAL;
    if (sp->M > MCB_MAX_M_APPLY) return MCB_EUNSUPPORTED;
    if (mode < MCB_AUTO || mode > MCB_SPARSE) return MCB_EINVAL;
    if (sp->M > MCB_MAX_M_TILED) {                                       // many orbitals: the generic path (mcb_apply_big.cu), or SPARSE
        if (mode == MCB_SPARSE) return 0;
        return (mode == MCB_AUTO || mode == MCB_GEMM) ? (sp->N >= 2 ? mcb_big_workspace_bytes(sp) : 0) : (long long)MCB_EUNSUPPORTED;
    }
    if (mode == MCB_SPARSE) return 0;
    mode = resolve_mode(sp, mode);
    if (mode == MCB_RUNS) return mcb_runs_supported(sp) ? mcb_runs_workspace_bytes(sp) : (long long)MCB_EUNSUPPORTED;
    if (mode != MCB_GEMM) return 0;
    return mcb_gemm_workspace_bytes(sp);
}

template <int M>
static int launch_direct(mcb_space* sp, bool use_maps, const mcb_c128* T, const mcb_c128* V,
                         const mcb_c128* d_C, mcb_c128* d_HC, cudaStream_t st)
{
    constexpr int P = M * (M + 1) / 2;
    // coefficients: T [M*M] complex, Vp [P*P] complex (interleaved)
    const size_t bytes = sizeof(mcb_c128) * (size_t)(M * M + P * P);
    if (mcb_coef_stale(sp)) {
        double* h = (double*)sp->h_coef;
        memcpy(h, T, sizeof(mcb_c128) * M * M);
        double* vr = h + 2 * (M * M + P * P);               // scratch behind the packed block
        double* vi = vr + P * P;
        mcb_pack_pairs(sp->N, M, T, V, false, vr, vi);
        for (int i = 0; i < P * P; ++i) { h[2 * (M * M + i)] = vr[i]; h[2 * (M * M + i) + 1] = vi[i]; }
        { int rc = mcb_coef_upload(sp, h, bytes, st); if (rc) return rc; }
        mcb_coef_staged(sp);
    }
    DirectArgs a;
    a.d = sp->dev; a.fock = sp->fock;
    a.C = (const double2*)d_C; a.HC = (double2*)d_HC; a.coef = (const double2*)sp->d_coef;
    a.map1 = sp->d_map1; a.ld1 = sp->map1_ld; a.map2 = sp->d_map2; a.ld2 = sp->map2_ld;
    const int threads = 128;
    const unsigned blocks = (unsigned)((sp->nc + threads - 1) / threads);
    { int rc = mcb_tick(sp, 0, st); if (rc) return rc; }
    if (use_maps) {
        MCB_CUDA(cudaFuncSetAttribute(k_hc_direct<M, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
        k_hc_direct<M, true><<<blocks, threads, bytes, st>>>(a);
    } else {
        MCB_CUDA(cudaFuncSetAttribute(k_hc_direct<M, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
        k_hc_direct<M, false><<<blocks, threads, bytes, st>>>(a);
    }
    MCB_CHECK_LAUNCH();
    { int rc = mcb_tick(sp, 1, st); if (rc) return rc; }
    mcb_tick_done(sp, 1);
    sp->last_launches = 1;
    return MCB_OK;
}

extern "C" int mcb_hc_apply(mcb_space* sp, const mcb_c128* T, const mcb_c128* V,
                            const mcb_c128* d_C, mcb_c128* d_HC, int mode, void* d_workspace, void* stream)
{
    if (!sp || !T || !V || !d_C || !d_HC) return MCB_EINVAL;
    if (mode < MCB_AUTO || mode > MCB_SPARSE) return MCB_EINVAL;
    if (sp->M > MCB_MAX_M_APPLY) return MCB_EUNSUPPORTED;
    if ((((uintptr_t)d_C) & 15) || (((uintptr_t)d_HC) & 15)) return MCB_EINVAL;
    {
        const char* c0 = (const char*)d_C; const char* h0 = (const char*)d_HC;
        const size_t len = (size_t)sp->nc * sizeof(mcb_c128);
        if (c0 < h0 + len && h0 < c0 + len) return MCB_EINVAL;          // overlap
    }
    cudaStream_t st = (cudaStream_t)stream;
    sp->n_memcpy = 0; sp->n_memset = 0;
    if (sp->M > MCB_MAX_M_TILED) {                                       // many orbitals: the generic path (mcb_apply_big.cu), or SPARSE
        if (mode == MCB_SPARSE || (mode == MCB_AUTO && sp->d_fock && mcb_sparse_preferred(sp, T, V))) {
            if (!sp->d_fock) return MCB_ENOTREADY;
            return mcb_launch_sparse(sp, T, V, d_C, d_HC, st);
        }
        if (mode != MCB_AUTO && mode != MCB_GEMM) return MCB_EUNSUPPORTED;
        if (sp->N >= 2) {
            if (!sp->d_fock) return MCB_ENOTREADY;
            if (!d_workspace || (((uintptr_t)d_workspace) & 255)) return MCB_EINVAL;
        }
        return mcb_launch_big(sp, T, V, d_C, d_HC, d_workspace, st);
    }
    if (!sp->d_fock) return MCB_ENOTREADY;
    if (mode == MCB_SPARSE || (mode == MCB_AUTO && mcb_sparse_preferred(sp, T, V)))
        return mcb_launch_sparse(sp, T, V, d_C, d_HC, st);
    mode = resolve_mode(sp, mode);
    if (mode == MCB_MAPS && (!sp->d_map1 || (sp->N >= 2 && !sp->d_map2))) {
        // no dense planes: the compact table (T folded into V) serves alone -- one structure, one kernel
        if (sp->d_map2c && sp->N >= 2) return mcb_launch_maps2c(sp, T, V, d_C, d_HC, st);
        return MCB_ENOTREADY;
    }
    if (mode == MCB_RUNS) {
        if (!mcb_runs_supported(sp)) return MCB_EUNSUPPORTED;
        if (!d_workspace || (((uintptr_t)d_workspace) & 255)) return MCB_EINVAL;
        return mcb_launch_runs(sp, T, V, d_C, d_HC, d_workspace, st);
    } else if (mode == MCB_GEMM) {
        if (!d_workspace || (((uintptr_t)d_workspace) & 255)) return MCB_EINVAL;
        return mcb_launch_gemm(sp, T, V, d_C, d_HC, d_workspace, st);
    } else {
        const bool use_maps = mode == MCB_MAPS;
        MCB_DISPATCH_APPLY_M(sp->M, return launch_direct<MT>(sp, use_maps, T, V, d_C, d_HC, st));
    }
    return MCB_EINVAL;
}

extern "C" int mcb_resolve_mode(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, int mode)
{
    if (!sp || !T || !V) return MCB_EINVAL;
    if (mode < MCB_AUTO || mode > MCB_SPARSE) return MCB_EINVAL;
    if (sp->M > MCB_MAX_M_APPLY) return MCB_EUNSUPPORTED;
    if (sp->M > MCB_MAX_M_TILED) {
        if (mode == MCB_SPARSE || (mode == MCB_AUTO && sp->d_fock && mcb_sparse_preferred(sp, T, V))) return MCB_SPARSE;
        return (mode == MCB_AUTO || mode == MCB_GEMM) ? MCB_GEMM : MCB_EUNSUPPORTED;
    }
    if (mode == MCB_SPARSE || (mode == MCB_AUTO && mcb_sparse_preferred(sp, T, V))) return MCB_SPARSE;
    return resolve_mode(sp, mode);
}

// Pipelined variant for MCB_RUNS: the contraction walks the intermediates in index order and an intermediate with top
// occupation j only gathers C inside the first nc - N_c(N-j-3, M) elements, so the kernel is launched at once and waits,
// segment by segment, for the prefix of C it needs while the host-to-device copy streams in on a second stream; the
// trailing sum writes HC straight into the (pinned, mapped) host vector.  H2D, compute and D2H overlap.
// (Measured at configs[2]: 7.3 ms for copy - apply - copy, 4.9 ms pipelined; copying finished pieces of HC back with
// host-issued DMA behind per-tile flags instead of the zero-copy stores: 5.8 ms.)
static int hc_apply_host_pipelined(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* h_C, mcb_c128* h_HC,
                                   mcb_c128* d_C_scratch, void* d_workspace, cudaStream_t st, bool* done)
{
    *done = false;
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, h_C) != cudaSuccess || at.type != cudaMemoryTypeHost) { cudaGetLastError(); return MCB_OK; }
    void* d_HC_mapped = nullptr;
    if (cudaHostGetDevicePointer(&d_HC_mapped, h_HC, 0) != cudaSuccess || !d_HC_mapped) { cudaGetLastError(); return MCB_OK; }
    if (!sp->copy_stream) {
        MCB_CUDA(cudaStreamCreateWithFlags(&sp->copy_stream, cudaStreamNonBlocking));
        MCB_CUDA(cudaEventCreateWithFlags(&sp->ev_a, cudaEventDisableTiming));
        MCB_CUDA(cudaEventCreateWithFlags(&sp->ev_b, cudaEventDisableTiming));
        MCB_CUDA(cudaHostAlloc((void**)&sp->h_prog, sizeof(int) * (MCB_H2D_CHUNKS + 4), cudaHostAllocDefault));
    }
    if (!d_workspace || (((uintptr_t)d_workspace) & 255)) return MCB_EINVAL;
    sp->h_prog[MCB_H2D_CHUNKS] = 0;
    int rc = mcb_launch_runs(sp, T, V, d_C_scratch, (mcb_c128*)d_HC_mapped, d_workspace, st, h_C);
    if (rc != MCB_OK) return rc;
    MCB_CUDA(cudaEventRecord(sp->ev_b, sp->copy_stream));
    MCB_CUDA(cudaStreamWaitEvent(st, sp->ev_b, 0));
    MCB_CUDA(cudaStreamSynchronize(st));
    *done = true;
    // the kernel gave up waiting for a piece of C: no CUDA call reported the failure, so record a code of our own choosing
    // (cudaErrorTimeout) for mcb_last_cuda_error() instead of leaving a stale one there
    if (sp->h_prog[MCB_H2D_CHUNKS] != 0) return mcb_set_cuda_error(cudaErrorTimeout);
    return MCB_OK;
}

// Pipelined variant for MCB_GEMM and MCB_SPARSE (M <= MCB_MAX_M_TILED): outputs and intermediates are cut into slabs by the
// occupation j of the last orbital, the most significant digit of the index order.  An output with n_{M-1} <= j gathers only
// from configurations with n_{M-1} <= j + 2, a PREFIX of C, and (GEMM) only from intermediates with m_{M-1} <= j; so slab k
// is computed as soon as its prefix of C is on the device, and its piece of HC goes back to the host while slab k + 1 computes.
// Three streams: copy-in (pieces of C, one event per slab), the caller's (kernels, waiting on those events), copy-out.
static int hc_apply_host_slabs(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* h_C, mcb_c128* h_HC,
                               int mode, mcb_c128* d_C, mcb_c128* d_HC, void* d_workspace, cudaStream_t st, bool* done)
{
    *done = false;
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, h_C) != cudaSuccess || at.type != cudaMemoryTypeHost) { cudaGetLastError(); return MCB_OK; }
    if (cudaPointerGetAttributes(&at, h_HC) != cudaSuccess || at.type != cudaMemoryTypeHost) { cudaGetLastError(); return MCB_OK; }
    if (sp->N < 2 || sp->nc < (1LL << 18)) return MCB_OK;                // too small to be worth three streams
    if (!sp->copy_stream) {
        MCB_CUDA(cudaStreamCreateWithFlags(&sp->copy_stream, cudaStreamNonBlocking));
        MCB_CUDA(cudaEventCreateWithFlags(&sp->ev_a, cudaEventDisableTiming));
        MCB_CUDA(cudaEventCreateWithFlags(&sp->ev_b, cudaEventDisableTiming));
        MCB_CUDA(cudaHostAlloc((void**)&sp->h_prog, sizeof(int) * (MCB_H2D_CHUNKS + 4), cudaHostAllocDefault));
    }
    if (!sp->out_stream) MCB_CUDA(cudaStreamCreateWithFlags(&sp->out_stream, cudaStreamNonBlocking));
    if (!sp->slabs_store) {
        sp->slabs_store = (McbSlabs*)calloc(1, sizeof(McbSlabs));
        if (!sp->slabs_store) return MCB_ENOMEM;
        for (int k = 0; k < MCB_MAX_SLABS; ++k) {
            MCB_CUDA(cudaEventCreateWithFlags(&sp->slabs_store->ev_in[k], cudaEventDisableTiming));
            MCB_CUDA(cudaEventCreateWithFlags(&sp->slabs_store->ev_out[k], cudaEventDisableTiming));
        }
    }
    McbSlabs* sl = sp->slabs_store;
    const int N = sp->N, M = sp->M, W = M + 1;
    // configurations of n particles with last occupation <= j: N_c(n, M) - N_c(n - j - 1, M)
    auto upto = [&](int n, int j) -> long long {
        const long long all = sp->h_binom[(size_t)n * W + M];
        return j >= n ? all : all - sp->h_binom[(size_t)(n - j - 1) * W + M];
    };
    // cut points: the smallest j whose outputs reach the next 1/MCB_MAX_SLABS of the space
    sl->n = 0;
    long long c_sent = 0;
    {
        // the kernels of this call wait for the events: order the copy-in stream behind what the caller's stream holds now
        MCB_CUDA(cudaEventRecord(sp->ev_a, st));
        MCB_CUDA(cudaStreamWaitEvent(sp->copy_stream, sp->ev_a, 0));
        MCB_CUDA(cudaStreamWaitEvent(sp->out_stream, sp->ev_a, 0));
    }
    for (int j = 0; j <= N && sl->n < MCB_MAX_SLABS; ++j) {
        const long long g1 = upto(N, j);
        const long long prev = sl->n ? sl->g_end[sl->n - 1] : 0;
        const bool last = g1 >= sp->nc || sl->n == MCB_MAX_SLABS - 1;
        if (!last && g1 - prev < sp->nc / MCB_MAX_SLABS) continue;
        const int k = sl->n++;
        sl->g_end[k] = last ? sp->nc : g1;
        // intermediates with last occupation <= j, rounded up to whole tiles of every tile size in use (64, 128)
        long long m1 = last ? sp->nc2 : upto(N - 2, j);
        m1 = (m1 + 127) / 128 * 128;
        if (m1 > sp->nc2) m1 = sp->nc2;
        sl->m_end[k] = m1;
        // the prefix of C the slab gathers from: last occupation of its last intermediate / output, plus two
        int jx = j;
        while (jx < N - 2 && upto(N - 2, jx) < m1) ++jx;
        long long need = last ? sp->nc : upto(N, jx + 2);
        if (need > sp->nc) need = sp->nc;
        if (need > c_sent) {
            MCB_CUDA(cudaMemcpyAsync(d_C + c_sent, h_C + c_sent, (size_t)(need - c_sent) * sizeof(mcb_c128), cudaMemcpyHostToDevice, sp->copy_stream));
            c_sent = need;
        }
        MCB_CUDA(cudaEventRecord(sl->ev_in[k], sp->copy_stream));
        if (last) break;
    }
    sp->slabs = sl;
    const int rc = mcb_hc_apply(sp, T, V, d_C, d_HC, mode, d_workspace, (void*)st);
    sp->slabs = NULL;
    if (rc != MCB_OK) { cudaStreamSynchronize(sp->copy_stream); cudaStreamSynchronize(st); return rc; }
    long long g0 = 0;
    for (int k = 0; k < sl->n; ++k) {
        MCB_CUDA(cudaStreamWaitEvent(sp->out_stream, sl->ev_out[k], 0));
        if (sl->g_end[k] > g0)
            MCB_CUDA(cudaMemcpyAsync(h_HC + g0, d_HC + g0, (size_t)(sl->g_end[k] - g0) * sizeof(mcb_c128), cudaMemcpyDeviceToHost, sp->out_stream));
        g0 = sl->g_end[k];
    }
    MCB_CUDA(cudaStreamSynchronize(sp->out_stream));
    MCB_CUDA(cudaStreamSynchronize(st));
    *done = true;
    return MCB_OK;
}

extern "C" int mcb_hc_apply_host(mcb_space* sp, const mcb_c128* T, const mcb_c128* V,
                                 const mcb_c128* h_C, mcb_c128* h_HC, int mode,
                                 mcb_c128* d_C_scratch, mcb_c128* d_HC_scratch, void* d_workspace, void* stream)
{
    if (!sp || !T || !V || !h_C || !h_HC || !d_C_scratch || !d_HC_scratch) return MCB_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t len = (size_t)sp->nc * sizeof(mcb_c128);
    if (sp->d_fock && sp->M <= MCB_MAX_M_APPLY && mode >= MCB_AUTO && mode <= MCB_SPARSE && h_C != h_HC &&
        mcb_resolve_mode(sp, T, V, mode) == MCB_RUNS && mcb_runs_supported(sp)) {
        bool done = false;
        int rc = hc_apply_host_pipelined(sp, T, V, h_C, h_HC, d_C_scratch, d_workspace, st, &done);
        if (rc != MCB_OK) return rc;
        if (done) return MCB_OK;                                         // else: vectors not pinned, take the plain path
    }
    if (sp->d_fock && sp->M <= MCB_MAX_M_TILED && mode >= MCB_AUTO && mode <= MCB_SPARSE && h_C != h_HC) {
        const int m = mcb_resolve_mode(sp, T, V, mode);
        if (m == MCB_GEMM || m == MCB_SPARSE) {
            bool done = false;
            int rc = hc_apply_host_slabs(sp, T, V, h_C, h_HC, mode, d_C_scratch, d_HC_scratch, d_workspace, st, &done);
            if (rc != MCB_OK) return rc;
            if (done) return MCB_OK;
        }
    }
    MCB_CUDA(cudaMemcpyAsync(d_C_scratch, h_C, len, cudaMemcpyHostToDevice, st));
    int rc = mcb_hc_apply(sp, T, V, d_C_scratch, d_HC_scratch, mode, d_workspace, stream);
    if (rc != MCB_OK) return rc;
    MCB_CUDA(cudaMemcpyAsync(h_HC, d_HC_scratch, len, cudaMemcpyDeviceToHost, st));
    MCB_CUDA(cudaStreamSynchronize(st));
    return MCB_OK;
}
