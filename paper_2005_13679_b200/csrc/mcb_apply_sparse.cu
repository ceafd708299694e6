// mcb_apply_sparse.cu -- MCB_SPARSE mode of hc_apply (Eq. 12-13) for STRUCTURED matrix elements
// (SURVEY.md 8(f) NEXT-4): Lieb-Liniger plane waves, where momentum conservation leaves 29 of the 225 packed
// two-body elements at M = 5 (BASELINE.json configs[1]), and the Bose-Hubbard case the paper names (PAPER.md:347:
// nearest-neighbour T, on-site V).
//
// One thread per output configuration g (the per-output gather form of MCB_REHASH), but the sums run over the
// NON-ZERO elements only:
//   * diagonal elements cost no gather at all:   T_kk n_k C_g   and   Vp[(ks)][(ks)] n_k (n_s - [k==s]) C_g
//     (remove k, s and put them back: the target is g itself) -- an on-site interaction is entirely of this kind;
//   * every other non-zero element (k,l) of T or ((k<=s),(q<=l)) of the packed V is one entry of a list that all
//     threads walk together (warp-uniform control flow): the target index follows from the prefix sums S_j,
//         index = nc - 1 - sum_{j=0}^{M-2} G[j][S_j + delta_j],   delta_j = -[j>=k] - [j>=s] + [j>=q] + [j>=l]   (mcb_device.cuh),
//     i.e. target = g + sum_j (G[j][S_j] - G[j][S_j + delta_j]): the host packs delta_j (3 bits per j) into the entry, the
//     thread keeps G[j][S_j] in registers and looks a table entry up only where delta_j != 0; the occupations the
//     amplitude needs are read from a per-thread column of shared memory (run-time orbital index, no local memory).
// Complex FMA accumulated in registers, no atomics.  With few non-zeros the path moves from FP64-bound toward the
// gather / HBM bound: per output 16 B of C per entry instead of P^2 products.
#include <string.h>
#include "mcb_device.cuh"

#define MCB_SPARSE_MAX_ENTRIES 1024

struct SparseArgs {
    McbDev d;
    McbFockView fock;
    const double2* C;
    double2* HC;
    const double2* coef;       // [M] T_kk, [P] Vp diagonal, [n1 + n2] entry values, then (as int) three index words per entry
    int n1, n2;                // off-diagonal entries of T, of the packed V
    int g0, g1;                // outputs [g0, g1) of this launch
};

template <int M>
__global__ void __launch_bounds__(128) k_hc_sparse(const SparseArgs p)
{
    constexpr int P = M * (M + 1) / 2;
    extern __shared__ double2 sp_coef[];                    // the coefficient block, then this CTA's occupations
    const int nent = p.n1 + p.n2;
    const int ncoef = M + P + nent;
    const int nwords = ncoef + (3 * nent + 3) / 4;          // + three index words per entry
    for (int i = threadIdx.x; i < nwords; i += blockDim.x) sp_coef[i] = p.coef[i];
    const double2* tdiag = sp_coef;
    const double2* vdiag = sp_coef + M;
    const double2* val = sp_coef + M + P;
    const int* idx = reinterpret_cast<const int*>(sp_coef + ncoef);
    int* occ_s = reinterpret_cast<int*>(sp_coef + nwords) + threadIdx.x;       // [M][128]: n_j of this thread at occ_s[j * 128]
    const McbDev& d = p.d;
    const int g = p.g0 + blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = g < p.g1;

    int S[M], G0[M];                                        // prefix sums and G[j][S_j]
    double dre = 0.0, dim = 0.0;
    {
        int n[M], run = 0;
#pragma unroll
        for (int j = 0; j < M; ++j) {
            n[j] = live ? (int)p.fock.occ[(long long)j * p.fock.ld + g] : 0;
            occ_s[j * 128] = n[j];
            run += n[j]; S[j] = run;
            G0[j] = (j + 1 < M) ? mcb_ldG(d.G, d.ldg, j, run) : 0;
        }
        __syncthreads();                                    // coefficient block staged (occupations are thread-private)
        // ---- diagonal: no gather ----
#pragma unroll
        for (int k = 0; k < M; ++k) { dre += tdiag[k].x * n[k]; dim += tdiag[k].y * n[k]; }
        int a = 0;
#pragma unroll
        for (int k = 0; k < M; ++k) {
#pragma unroll
            for (int s = k; s < M; ++s, ++a) {
                const double f = (double)(n[k] * (n[s] - (k == s ? 1 : 0)));
                dre += vdiag[a].x * f; dim += vdiag[a].y * f;
            }
        }
    }
    if (!live) return;
    const double2 cg = p.C[g];
    double2 acc = make_double2(dre * cg.x - dim * cg.y, dre * cg.y + dim * cg.x);

    // ---- off-diagonal entries: one gather each.  Entry words: (k, s, q, l) bytes; then 3 bits per orbital j < M - 1
    //      with 2 + delta_j, delta_j = -[j>=k] - [j>=s] + [j>=q] + [j>=l] the change of the prefix sum S_j: the target is
    //      g + sum_j (G[j][S_j] - G[j][S_j + delta_j]), a look-up only where delta_j != 0 (uniform over the CTA) ----
#pragma unroll 1
    for (int e = 0; e < nent; ++e) {
        const int w = idx[3 * e];
        const int k = w & 255, s = (w >> 8) & 255, q = (w >> 16) & 255, l = (w >> 24) & 255;     // one-body: s = q = k (unused)
        const bool two = e >= p.n1;
        const int nk = occ_s[k * 128], nl = occ_s[l * 128];
        double amp;
        if (two) {
            const int ns = occ_s[s * 128], nq = occ_s[q * 128];
            const bool ok = (k == s) ? (nk >= 2) : (nk >= 1 && ns >= 1);
            if (!ok) continue;
            const int mq = nq - (q == k) - (q == s), ml = nl - (l == k) - (l == s);
            const double f1 = (k == s) ? __ldg(d.sq2 + nk) : __ldg(d.sq + nk) * __ldg(d.sq + ns);
            const double f2 = (q == l) ? __ldg(d.sq2 + mq + 2) : __ldg(d.sq + mq + 1) * __ldg(d.sq + ml + 1);
            amp = f1 * f2;
        } else {
            if (nk < 1) continue;
            amp = __ldg(d.sq + nk) * __ldg(d.sq + nl + 1);
        }
        int tgt = g;
        {
            const int wlo = idx[3 * e + 1], whi = idx[3 * e + 2];
#pragma unroll
            for (int j = 0; j + 1 < M; ++j) {
                const int dj = (((j < 10 ? wlo >> (3 * j) : whi >> (3 * (j - 10))) & 7)) - 2;
                if (dj != 0) tgt += G0[j] - mcb_ldG(d.G, d.ldg, j, S[j] + dj);
            }
        }
        const double2 z = __ldg(p.C + MCB_CHK(p.d, tgt, p.d.nc, 501));
        const double2 v = val[e];
        const double zr = amp * z.x, zi = amp * z.y;
        acc.x = fma(v.x, zr, acc.x); acc.x = fma(-v.y, zi, acc.x);
        acc.y = fma(v.x, zi, acc.y); acc.y = fma(v.y, zr, acc.y);
    }
    p.HC[g] = acc;
}

// =========================================================================================================
// host
// =========================================================================================================
// Packs T and the bosonic-symmetric part of V (mcb_pack_pairs, no folding) into the diagonal tables and the entry
// list.  Returns the number of off-diagonal entries (n1 + n2), or -1 if the list does not fit.
// index words of one entry: orbitals as bytes (one-body: s = q = k, never used), then 2 + delta_j in 3 bits per j
static void sparse_words(int M, int k, int s, int q, int l, int* w)
{
    const bool two = s >= 0;
    w[0] = k | ((two ? s : k) << 8) | ((two ? q : k) << 16) | (l << 24);
    unsigned long long bits = 0;
    for (int j = 0; j + 1 < M; ++j) {
        int dj = -(j >= k ? 1 : 0) + (j >= l ? 1 : 0);
        if (two) dj += -(j >= s ? 1 : 0) + (j >= q ? 1 : 0);
        const unsigned long long f = (unsigned long long)(dj + 2);
        if (j < 10) bits |= f << (3 * j); else bits |= f << (32 + 3 * (j - 10));
    }
    w[1] = (int)(unsigned)(bits & 0xffffffffull);
    w[2] = (int)(unsigned)(bits >> 32);
}

static int sparse_pack(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, int* n1_out, int* n2_out, size_t* bytes_out, bool count_only)
{
    const int M = sp->M, P = sp->P;
    double* vr = (double*)((char*)sp->h_coef + sp->coef_bytes) - 2 * (size_t)P * P;          // scratch at the end of h_coef
    double* vi = vr + (size_t)P * P;
    mcb_pack_pairs(sp->N, M, T, V, false, vr, vi);
    int n1 = 0, n2 = 0;
    for (int k = 0; k < M; ++k)
        for (int l = 0; l < M; ++l)
            if (k != l && (T[k * M + l].re != 0.0 || T[k * M + l].im != 0.0)) ++n1;
    if (sp->N >= 2)
        for (int a = 0; a < P; ++a)
            for (int c = 0; c < P; ++c)
                if (a != c && (vr[a * P + c] != 0.0 || vi[a * P + c] != 0.0)) ++n2;
    *n1_out = n1; *n2_out = n2;
    const int nent = n1 + n2;
    const size_t bytes = sizeof(double) * 2 * (size_t)(M + P + nent) + sizeof(double) * 2 * (size_t)((3 * nent + 3) / 4);
    *bytes_out = bytes;
    if (nent > MCB_SPARSE_MAX_ENTRIES || bytes + 2 * sizeof(double) * (size_t)P * P > sp->coef_bytes) return -1;
    if (count_only) return nent;
    double* h = (double*)sp->h_coef;
    for (int k = 0; k < M; ++k) { h[2 * k] = T[k * M + k].re; h[2 * k + 1] = T[k * M + k].im; }
    for (int a = 0; a < P; ++a) {
        const bool on = sp->N >= 2;
        h[2 * (M + a)] = on ? vr[a * P + a] : 0.0; h[2 * (M + a) + 1] = on ? vi[a * P + a] : 0.0;
    }
    double* val = h + 2 * (M + P);
    int* idx = (int*)(val + 2 * (size_t)nent);
    int e = 0;
    for (int k = 0; k < M; ++k)
        for (int l = 0; l < M; ++l)
            if (k != l && (T[k * M + l].re != 0.0 || T[k * M + l].im != 0.0)) {
                val[2 * e] = T[k * M + l].re; val[2 * e + 1] = T[k * M + l].im;
                sparse_words(M, k, -1, -1, l, idx + 3 * e); ++e;
            }
    if (sp->N >= 2) {
        int a = 0;
        for (int k = 0; k < M; ++k)
            for (int s = k; s < M; ++s, ++a) {
                int c = 0;
                for (int q = 0; q < M; ++q)
                    for (int l = q; l < M; ++l, ++c)
                        if (a != c && (vr[a * P + c] != 0.0 || vi[a * P + c] != 0.0)) {
                            val[2 * e] = vr[a * P + c]; val[2 * e + 1] = vi[a * P + c];
                            sparse_words(M, k, s, q, l, idx + 3 * e); ++e;
                        }
            }
    }
    return nent;
}

// off-diagonal fill of the packed V small enough for the sparse path to win (used by MCB_AUTO)
bool mcb_sparse_preferred(mcb_space* sp, const mcb_c128* T, const mcb_c128* V)
{
    int n1, n2; size_t bytes;
    if (sp->M > MCB_MAX_M_TILED) return false;
    if (sparse_pack(sp, T, V, &n1, &n2, &bytes, true) < 0) return false;
    return 4 * (long long)n2 <= (long long)sp->P * sp->P;             // the M (M - 1) one-body entries never dominate
}

template <int M>
static int launch_sparse_m(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_C, mcb_c128* d_HC, cudaStream_t st)
{
    int n1, n2; size_t bytes;
    if (mcb_coef_stale(sp)) {
        if (sparse_pack(sp, T, V, &n1, &n2, &bytes, false) < 0) return MCB_EUNSUPPORTED;
        { int rc = mcb_coef_upload(sp, sp->h_coef, bytes, st); if (rc) return rc; }
        sp->hold_n1 = n1; sp->hold_n2 = n2; sp->hold_bytes = bytes;
        mcb_coef_staged(sp);
    } else { n1 = sp->hold_n1; n2 = sp->hold_n2; bytes = sp->hold_bytes; }
    SparseArgs a;
    a.d = sp->dev; a.fock = sp->fock; a.C = (const double2*)d_C; a.HC = (double2*)d_HC;
    a.coef = (const double2*)sp->d_coef; a.n1 = n1; a.n2 = n2;
    const int threads = 128;
    const size_t smem = bytes + sizeof(int) * (size_t)M * 128;          // + the CTA's occupations
    if (smem > sp->sparse_smem_set) {                                    // per space (per device); grows with the entry list only
        MCB_CUDA(cudaFuncSetAttribute(k_hc_sparse<M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        sp->sparse_smem_set = smem;
    }
    if (sp->slabs) {
        // pipelined host apply: one launch per slab of outputs, each behind the arrival of the prefix of C it gathers from
        long long g0 = 0;
        for (int k = 0; k < sp->slabs->n; ++k) {
            const long long g1 = sp->slabs->g_end[k];
            MCB_CUDA(cudaStreamWaitEvent(st, sp->slabs->ev_in[k], 0));
            if (g1 > g0) {
                a.g0 = (int)g0; a.g1 = (int)g1;
                k_hc_sparse<M><<<(unsigned)((g1 - g0 + threads - 1) / threads), threads, smem, st>>>(a);
                MCB_CHECK_LAUNCH();
            }
            MCB_CUDA(cudaEventRecord(sp->slabs->ev_out[k], st));
            g0 = g1;
        }
        sp->last_launches = sp->slabs->n;
        return MCB_OK;
    }
    const unsigned blocks = (unsigned)((sp->nc + threads - 1) / threads);
    a.g0 = 0; a.g1 = (int)sp->nc;
    { int rc = mcb_tick(sp, 0, st); if (rc) return rc; }
    k_hc_sparse<M><<<blocks, threads, smem, st>>>(a);
    MCB_CHECK_LAUNCH();
    { int rc = mcb_tick(sp, 1, st); if (rc) return rc; }
    mcb_tick_done(sp, 1);
    sp->last_launches = 1;
    return MCB_OK;
}

int mcb_launch_sparse(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_C, mcb_c128* d_HC, cudaStream_t st)
{
    switch (sp->M) {
    case 1: return launch_sparse_m<1>(sp, T, V, d_C, d_HC, st);
    case 2: return launch_sparse_m<2>(sp, T, V, d_C, d_HC, st);
    case 3: return launch_sparse_m<3>(sp, T, V, d_C, d_HC, st);
    case 4: return launch_sparse_m<4>(sp, T, V, d_C, d_HC, st);
    case 5: return launch_sparse_m<5>(sp, T, V, d_C, d_HC, st);
    case 6: return launch_sparse_m<6>(sp, T, V, d_C, d_HC, st);
    case 7: return launch_sparse_m<7>(sp, T, V, d_C, d_HC, st);
    case 8: return launch_sparse_m<8>(sp, T, V, d_C, d_HC, st);
    case 9: return launch_sparse_m<9>(sp, T, V, d_C, d_HC, st);
    case 10: return launch_sparse_m<10>(sp, T, V, d_C, d_HC, st);
    case 11: return launch_sparse_m<11>(sp, T, V, d_C, d_HC, st);
    case 12: return launch_sparse_m<12>(sp, T, V, d_C, d_HC, st);
    default: return MCB_EUNSUPPORTED;
    }
}
