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
//     threads walk together (warp-uniform control flow).  NOTHING about an entry is decoded on the device: the host
//     turns it into a descriptor of shared-memory row numbers, and each thread prepares, once, the few numbers of ITS
//     configuration any entry can ask for:
//       amplitude:  every amplitude of Eq. 12-13 is a product of at most four factors sqrt(n_j + c), c in {-1, 0, 1, 2}
//                   (remove k, s: sqrt(n_k) sqrt(n_s - [k==s]); insert q, l into m = n - e_k - e_s: sqrt(m_q + 1)
//                   sqrt(m_l + 1 + [q==l])) -- the thread keeps the 4 M values R[4 j + c + 1] = sqrt(n_j + c) (and a row of
//                   ones) in its column of shared memory; a removal that is not allowed makes one factor sqrt(0) = 0;
//       target:     index = nc - 1 - sum_{j=0}^{M-2} G[j][S_j]  (mcb_device.cuh), so the target of an entry that shifts the
//                   prefix sum S_j by delta_j = -[j>=k] - [j>=s] + [j>=q] + [j>=l] is
//                       g + sum_j (G[j][S_j] - G[j][S_j + delta_j]);
//                   the j = 0 term is -delta_0 (G[0][x] = x: a constant of the entry), and for j >= 1 the thread keeps the
//                   4 (M - 2) differences D[4 (j - 1) + code(delta)] for delta in {-2, -1, 1, 2} in its column.
//     Per entry and thread that leaves: one descriptor (broadcast), four factor loads, the D rows with delta_j != 0, one
//     16-byte gather of C (skipped when the amplitude is 0) and the complex multiply-add.
// Complex FMA accumulated in registers, no atomics.  With few non-zeros the path moves from FP64-bound toward the
// gather / HBM bound: per output 16 B of C per entry instead of P^2 products.
#include <string.h>
#include "mcb_device.cuh"

#define MCB_SPARSE_MAX_ENTRIES 1024
#define SPARSE_THREADS 128

struct SparseArgs {
    McbDev d;
    McbFockView fock;
    const double2* C;
    double2* HC;
    const double2* coef;       // [M] T_kk, [P] Vp diagonal, [nent] entry values, [nent] descriptors (int4), [nent] int (more D rows)
    int n1, n2;                // off-diagonal entries of T, of the packed V
    int g0, g1;                // outputs [g0, g1) of this launch
};

// 16-byte units of the staged coefficient block
__host__ __device__ inline int sparse_block_units(int M, int nent) { return M + M * (M + 1) / 2 + 2 * nent + (nent + 3) / 4; }
template <int M> struct SparseCfg {
    static constexpr int RROWS = 4 * M + 1;                              // sqrt(n_j + c) rows + the row of ones
    static constexpr int DROWS = M > 2 ? 4 * (M - 2) : 0;                // index differences, j = 1 .. M - 2
    static constexpr size_t PER_CTA = (size_t)SPARSE_THREADS * (RROWS * sizeof(double) + DROWS * sizeof(int));
};

template <int M>
__global__ void __launch_bounds__(SPARSE_THREADS) k_hc_sparse(const SparseArgs p)
{
    constexpr int P = M * (M + 1) / 2;
    using Cfg = SparseCfg<M>;
    extern __shared__ double2 sp_coef[];                    // the coefficient block, then the per-thread columns
    const int nent = p.n1 + p.n2;
    const int nunits = sparse_block_units(M, nent);
    for (int i = threadIdx.x; i < nunits; i += SPARSE_THREADS) sp_coef[i] = p.coef[i];
    const double2* tdiag = sp_coef;
    const double2* vdiag = sp_coef + M;
    const double2* val = sp_coef + M + P;
    const int4* desc = reinterpret_cast<const int4*>(sp_coef + M + P + nent);
    const int* more = reinterpret_cast<const int*>(sp_coef + M + P + 2 * nent);
    double* R = reinterpret_cast<double*>(sp_coef + nunits) + threadIdx.x;               // R[row * 128]
    int* D = reinterpret_cast<int*>(reinterpret_cast<double*>(sp_coef + nunits) + Cfg::RROWS * SPARSE_THREADS) + threadIdx.x;
    const McbDev& d = p.d;
    const int g = p.g0 + blockIdx.x * SPARSE_THREADS + threadIdx.x;
    const bool live = g < p.g1;

    double dre = 0.0, dim = 0.0;
    {
        int n[M], run = 0;
#pragma unroll
        for (int j = 0; j < M; ++j) {
            n[j] = live ? (int)p.fock.occ[(long long)j * p.fock.ld + g] : 0;
            run += n[j];
#pragma unroll
            for (int c = -1; c <= 2; ++c) R[(4 * j + c + 1) * SPARSE_THREADS] = __ldg(d.sq + max(n[j] + c, 0));
            if (j >= 1 && j + 1 < M) {
                const int g0j = mcb_ldG(d.G, d.ldg, j, run);
#pragma unroll
                for (int code = 0; code < 4; ++code) {
                    const int t = run + (code < 2 ? code - 2 : code - 1);                // delta = -2, -1, +1, +2
                    D[(4 * (j - 1) + code) * SPARSE_THREADS] = (t >= 0 && t <= d.N) ? g0j - mcb_ldG(d.G, d.ldg, j, t) : 0;
                }
            }
        }
        R[4 * M * SPARSE_THREADS] = 1.0;
        __syncthreads();                                    // coefficient block staged (the columns are thread-private)
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

    // ---- off-diagonal entries: descriptor = (two factor rows | two factor rows | 2 - delta_0 and the number of D rows |
    //      five D rows of 6 bits); rows are pre-multiplied by the column stride where they fit ----
#pragma unroll 2
    for (int e = 0; e < nent; ++e) {
        const int4 ds = desc[e];
        const double amp = (R[ds.x & 0xffff] * R[(unsigned)ds.x >> 16]) * (R[ds.y & 0xffff] * R[(unsigned)ds.y >> 16]);
        int tgt = g + (ds.z & 7) - 2;
        const int ng = ds.z >> 3;
#pragma unroll
        for (int t = 0; t < M - 2; ++t) {
            if (t < ng) {
                const int w = t < 5 ? ds.w : more[e];
                tgt += D[((w >> (6 * (t % 5))) & 63) * SPARSE_THREADS];
            }
        }
        double2 z = make_double2(0.0, 0.0);
        if (amp != 0.0) z = __ldg(p.C + MCB_CHK(p.d, tgt, p.d.nc, 501));
        const double2 v = val[e];
        const double zr = amp * z.x, zi = amp * z.y;
        acc.x = fma(v.x, zr, acc.x); acc.x = fma(-v.y, zi, acc.x);
        acc.y = fma(v.x, zi, acc.y); acc.y = fma(v.y, zr, acc.y);
    }
    p.HC[g] = acc;
}

// ---- many orbitals (12 < M <= 32; a Bose-Hubbard lattice is naturally larger than 12 sites): the same kernel with
// M a run-time value.  64 threads per CTA (the columns of a thread take 4 M + 1 doubles and 5 M - 8 ints: 113 KB per CTA at
// M = 32), the occupations kept in the thread's column for the diagonal sums, and the D rows of an entry listed as bytes
// (up to M - 2 = 30 of them, 32 bytes per entry) instead of 6-bit fields.
#define SPARSE_RT_THREADS 64
__host__ __device__ inline int sparse_rt_block_units(int M, int nent) { return M + M * (M + 1) / 2 + 4 * nent; }
static size_t sparse_rt_per_cta(int M)
{
    return (size_t)SPARSE_RT_THREADS * ((4 * M + 1) * sizeof(double) + (4 * (M - 2) + M) * sizeof(int));
}

__global__ void __launch_bounds__(SPARSE_RT_THREADS) k_hc_sparse_rt(const SparseArgs p)
{
    const McbDev& d = p.d;
    const int M = d.M, P = M * (M + 1) / 2;
    extern __shared__ double2 sp_coef[];
    const int nent = p.n1 + p.n2;
    const int nunits = sparse_rt_block_units(M, nent);
    for (int i = threadIdx.x; i < nunits; i += SPARSE_RT_THREADS) sp_coef[i] = p.coef[i];
    const double2* tdiag = sp_coef;
    const double2* vdiag = sp_coef + M;
    const double2* val = sp_coef + M + P;
    const int4* desc = reinterpret_cast<const int4*>(sp_coef + M + P + nent);
    const unsigned char* rows = reinterpret_cast<const unsigned char*>(sp_coef + M + P + 2 * nent);      // [nent][32]
    double* R = reinterpret_cast<double*>(sp_coef + nunits) + threadIdx.x;                               // R[row * 64]
    int* D = reinterpret_cast<int*>(reinterpret_cast<double*>(sp_coef + nunits) + (4 * M + 1) * SPARSE_RT_THREADS) + threadIdx.x;
    int* Nn = D + 4 * (M - 2) * SPARSE_RT_THREADS;                                                      // Nn[j * 64]
    const int g = p.g0 + blockIdx.x * SPARSE_RT_THREADS + threadIdx.x;
    const bool live = g < p.g1;
    {
        int run = 0;
        for (int j = 0; j < M; ++j) {
            const int nj = live ? (int)p.fock.occ[(long long)j * p.fock.ld + g] : 0;
            Nn[j * SPARSE_RT_THREADS] = nj;
            run += nj;
#pragma unroll
            for (int c = -1; c <= 2; ++c) R[(4 * j + c + 1) * SPARSE_RT_THREADS] = __ldg(d.sq + max(nj + c, 0));
            if (j >= 1 && j + 1 < M) {
                const int g0j = mcb_ldG(d.G, d.ldg, j, run);
#pragma unroll
                for (int code = 0; code < 4; ++code) {
                    const int t = run + (code < 2 ? code - 2 : code - 1);
                    D[(4 * (j - 1) + code) * SPARSE_RT_THREADS] = (t >= 0 && t <= d.N) ? g0j - mcb_ldG(d.G, d.ldg, j, t) : 0;
                }
            }
        }
        R[4 * M * SPARSE_RT_THREADS] = 1.0;
    }
    __syncthreads();
    if (!live) return;
    double dre = 0.0, dim = 0.0;
    {
        int a = 0;
        for (int k = 0; k < M; ++k) {
            const int nk = Nn[k * SPARSE_RT_THREADS];
            dre += tdiag[k].x * nk; dim += tdiag[k].y * nk;
            if (nk == 0) { a += M - k; continue; }                       // every pair (k, s) of an empty orbital k contributes 0
            for (int s = k; s < M; ++s, ++a) {
                const double f = (double)(nk * (Nn[s * SPARSE_RT_THREADS] - (k == s ? 1 : 0)));
                dre += vdiag[a].x * f; dim += vdiag[a].y * f;
            }
        }
    }
    const double2 cg = p.C[g];
    double2 acc = make_double2(dre * cg.x - dim * cg.y, dre * cg.y + dim * cg.x);
#pragma unroll 1
    for (int e = 0; e < nent; ++e) {
        const int4 ds = desc[e];
        const double amp = (R[ds.x & 0xffff] * R[(unsigned)ds.x >> 16]) * (R[ds.y & 0xffff] * R[(unsigned)ds.y >> 16]);
        if (amp == 0.0) continue;
        int tgt = g + (ds.z & 7) - 2;
        const int ng = ds.z >> 3;
        const unsigned char* rw = rows + 32 * e;
        for (int t = 0; t < ng; ++t) tgt += D[(int)rw[t] * SPARSE_RT_THREADS];
        const double2 z = __ldg(p.C + MCB_CHK(p.d, tgt, p.d.nc, 502));
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
// Descriptor of one entry (see the kernel): one-body entries have s = q = -1.
// (M > MCB_MAX_M_TILED: column stride of k_hc_sparse_rt, and the D rows as bytes in rows32[32] instead of the 6-bit fields)
static void sparse_desc(int M, int k, int s, int q, int l, int* d4, int* more, unsigned char* rows32)
{
    const bool two = s >= 0;
    const int ONE = 4 * M;                                               // the row of ones
    const int STRIDE = rows32 ? SPARSE_RT_THREADS : SPARSE_THREADS;
    auto row = [&](int j, int c) { return (4 * j + c + 1) * STRIDE; };
    int f[4];
    f[0] = row(k, 0);                                                    // sqrt(n_k)
    if (two) {
        f[1] = row(s, k == s ? -1 : 0);                                  // sqrt(n_s - [k==s])
        f[2] = row(q, 1 - (q == k) - (q == s));                          // sqrt(m_q + 1),  m = n - e_k - e_s
        f[3] = row(l, 1 - (l == k) - (l == s) + (q == l));               // sqrt(m_l + 1 + [q==l])
    } else {
        f[1] = row(l, 1);                                                // sqrt(n_l + 1)   (k != l)
        f[2] = ONE * STRIDE; f[3] = ONE * STRIDE;
    }
    d4[0] = f[0] | (f[1] << 16);
    d4[1] = f[2] | (f[3] << 16);
    int ng = 0, delta0 = 0;
    unsigned long long bits = 0;
    for (int j = 0; j + 1 < M; ++j) {
        int dj = -(j >= k ? 1 : 0) + (j >= l ? 1 : 0);
        if (two) dj += -(j >= s ? 1 : 0) + (j >= q ? 1 : 0);
        if (j == 0) { delta0 = dj; continue; }
        if (dj == 0) continue;
        const int code = dj < 0 ? dj + 2 : dj + 1;                       // -2, -1, +1, +2 -> 0, 1, 2, 3
        const unsigned long long r = (unsigned long long)(4 * (j - 1) + code);
        if (rows32) rows32[ng] = (unsigned char)r;
        else if (ng < 5) bits |= r << (6 * ng); else bits |= r << (32 + 6 * (ng - 5));
        ++ng;
    }
    d4[2] = (2 - delta0) | (ng << 3);                                    // target = g - delta_0 + sum of the D rows
    d4[3] = (int)(unsigned)(bits & 0xffffffffull);
    if (more) *more = (int)(unsigned)(bits >> 32);
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
    const bool rt = M > MCB_MAX_M_TILED;
    const size_t bytes = sizeof(double) * 2 * (size_t)(rt ? sparse_rt_block_units(M, nent) : sparse_block_units(M, nent));
    *bytes_out = bytes;
    if (nent > MCB_SPARSE_MAX_ENTRIES || bytes + 2 * sizeof(double) * (size_t)P * P > sp->coef_bytes) return -1;
    if (count_only) return nent;
    double* h = (double*)sp->h_coef;
    memset(h, 0, bytes);
    for (int k = 0; k < M; ++k) { h[2 * k] = T[k * M + k].re; h[2 * k + 1] = T[k * M + k].im; }
    for (int a = 0; a < P; ++a) {
        const bool on = sp->N >= 2;
        h[2 * (M + a)] = on ? vr[a * P + a] : 0.0; h[2 * (M + a) + 1] = on ? vi[a * P + a] : 0.0;
    }
    double* val = h + 2 * (M + P);
    int* desc = (int*)(val + 2 * (size_t)nent);
    int* more = desc + 4 * (size_t)nent;
    unsigned char* rows32 = (unsigned char*)more;                        // run-time-M layout: 32 bytes per entry behind the descriptors
    int e = 0;
    for (int k = 0; k < M; ++k)
        for (int l = 0; l < M; ++l)
            if (k != l && (T[k * M + l].re != 0.0 || T[k * M + l].im != 0.0)) {
                val[2 * e] = T[k * M + l].re; val[2 * e + 1] = T[k * M + l].im;
                if (rt) sparse_desc(M, k, -1, -1, l, desc + 4 * e, nullptr, rows32 + 32 * (size_t)e);
                else sparse_desc(M, k, -1, -1, l, desc + 4 * e, more + e, nullptr);
                ++e;
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
                            if (rt) sparse_desc(M, k, s, q, l, desc + 4 * e, nullptr, rows32 + 32 * (size_t)e);
                            else sparse_desc(M, k, s, q, l, desc + 4 * e, more + e, nullptr);
                            ++e;
                        }
            }
    }
    return nent;
}

// off-diagonal fill of the packed V small enough for the sparse path to win (used by MCB_AUTO)
bool mcb_sparse_preferred(mcb_space* sp, const mcb_c128* T, const mcb_c128* V)
{
    int n1, n2; size_t bytes;
    if (sp->M > MCB_MAX_M_TILED && sp->N < 2) return false;             // (one particle, many orbitals: the M x M mat-vec needs no table)
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
    const int threads = SPARSE_THREADS;
    const size_t smem = bytes + SparseCfg<M>::PER_CTA;                   // + the threads' columns of factors and index differences
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

static int launch_sparse_rt(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_C, mcb_c128* d_HC, cudaStream_t st)
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
    a.g0 = 0; a.g1 = (int)sp->nc;
    const size_t smem = bytes + sparse_rt_per_cta(sp->M);
    if (smem > 227 * 1024) return MCB_EUNSUPPORTED;
    if (smem > sp->sparse_smem_set) {
        MCB_CUDA(cudaFuncSetAttribute(k_hc_sparse_rt, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        sp->sparse_smem_set = smem;
    }
    { int rc = mcb_tick(sp, 0, st); if (rc) return rc; }
    k_hc_sparse_rt<<<(unsigned)((sp->nc + SPARSE_RT_THREADS - 1) / SPARSE_RT_THREADS), SPARSE_RT_THREADS, smem, st>>>(a);
    MCB_CHECK_LAUNCH();
    { int rc = mcb_tick(sp, 1, st); if (rc) return rc; }
    mcb_tick_done(sp, 1);
    sp->last_launches = 1;
    return MCB_OK;
}

int mcb_launch_sparse(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_C, mcb_c128* d_HC, cudaStream_t st)
{
    if (sp->M > MCB_MAX_M_TILED) return launch_sparse_rt(sp, T, V, d_C, d_HC, st);
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
