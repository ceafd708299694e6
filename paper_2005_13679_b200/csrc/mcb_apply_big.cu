// mcb_apply_big.cu -- hc_apply and the density matrices for MANY orbitals (12 < M <= 32): the paper's second sweep, N = 5
// particles with M up to 25 orbitals, and its ground-state runs N = 5, M = 11 and 21.
//
// The packed coefficient matrix Vp (P x P complex, P = M(M+1)/2 up to 528: 4.5 MB) no longer fits on chip, M is a run-time
// value, and the (N-2)-particle space is small when N is small (N = 5, M = 21: nc = 53,130 but nc2 = 1,771).  Same
// factorisation through the (N-2)-particle space as MCB_GEMM (mcb_apply_gemm.cu), written for generality:
//   k_big_contract W'[a][m] = F(m,a) sum_c Vp[a][c] F(m,c) C[index(m + e_q + e_l)] (index = nc - 1 - X[q] - Y[l],
//                  mcb_device.cuh): the real 2P x 2P x nc2 product on mma.sync.m8n8k4.f64, 64 x 64 complex tiles, Vp streamed
//                  from L2 and the gather of C fused into the B-tile load -- the workspace holds W' only (P x nc2 complex);
//   k_big_gather   D[c][m] = F(m,c) C[index(m + e_q + e_l)] materialised (P x nc2 complex): the density matrices only;
//   k_big_reduce   HC[g] = sum over the allowed removal pairs a of W'[a][index2(n^g - e_k - e_s)] -- every W' element is
//                  read by exactly one g: no atomics.  T rides inside Vp (sum_s a+_s a_s = N), as in MCB_GEMM.
//   k_big_gram     G[a][c] = sum_m conj(D[a][m]) D[c][m] (split over m, fixed-order finish): rho2 = G, rho1 from the number
//                  operator -- mcb_rho for M > 12; mcb_lanczos inherits the apply.
//   N = 1 (no (N-2)-particle space): HC = T.C, a plain M x M mat-vec (k_big_onebody).
#include <stdlib.h>
#include <string.h>
#include "mcb_device.cuh"

#define BIG_THREADS 128
#define BIG_SPLIT_MAX 64              // partial Gram matrices

struct BigArgs {
    McbDev d;
    McbFockView fock;
    const double2* C;
    double2* HC;
    const double2* Vp;         // [P][P] row-major, T folded in
    double2* D;                // [P][ld2]
    double2* W;                // [P][ld2]
    long long ld2;
    int P;
};

// prefix sums -> X[q], Y[l] of the double jump from an intermediate (mcb_maps.cu k_map2 has the derivation); run-time M
__device__ __forceinline__ void big_xy(const McbDev& d, const int* S, int* X, int* Y)
{
    const int M = d.M;
    int x = 0, tot1 = 0;
    int A1[MCB_MAX_M], A2[MCB_MAX_M];
    for (int j = 0; j < M; ++j) {
        X[j] = x;
        if (j <= M - 2) {
            const int a0 = mcb_ldG(d.G, d.ldg, j, S[j]);
            A1[j] = mcb_ldG(d.G, d.ldg, j, S[j] + 1);
            A2[j] = mcb_ldG(d.G, d.ldg, j, S[j] + 2);
            x += a0 - A1[j]; tot1 += A1[j];
        } else { A1[j] = 0; A2[j] = 0; }
    }
    int pre = tot1, suf = 0;
    for (int l = M - 1; l >= 0; --l) { pre -= A1[l]; suf += A2[l]; Y[l] = pre + suf; }
}

__global__ void __launch_bounds__(BIG_THREADS) k_big_gather(const BigArgs p)
{
    const McbDev& d = p.d;
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= d.nc2) return;
    const int M = d.M;
    int S[MCB_MAX_M], X[MCB_MAX_M], Y[MCB_MAX_M];
    double r1[MCB_MAX_M], r2[MCB_MAX_M];
    int run = 0;
    for (int j = 0; j < M; ++j) {
        const int nj = (int)p.fock.occ2[(long long)j * p.fock.ld2 + m];
        run += nj; S[j] = run;
        r1[j] = __ldg(d.sq + nj + 1);
        r2[j] = __ldg(d.sq2 + nj + 2);
    }
    big_xy(d, S, X, Y);
    const int base = d.nc - 1;
    int c = 0;
    for (int q = 0; q < M; ++q)
        for (int l = q; l < M; ++l, ++c) {
            const double2 z = __ldg(p.C + MCB_CHK(d, base - X[q] - Y[l], d.nc, 201));
            const double f = (q == l) ? r2[q] : r1[q] * r1[l];
            p.D[(long long)c * p.ld2 + m] = make_double2(f * z.x, f * z.y);
        }
}

// ---- the contraction on the FP64 tensor path, with the gather fused into the B-tile load (no materialised D) ----------------
// W'[a][m] = F(m,a) sum_c Vp[a][c] F(m,c) C[index(m + e_q + e_l)] as the REAL product
//     [Re W; Im W] = [[Re Vp, -Im Vp], [Im Vp, Re Vp]] [Re D; Im D]         (2P x 2P times 2P x nc2)
// on mma.sync.m8n8k4.f64.  CTA tile: CT_BM = 64 rows a (128 real rows: the 64 real parts, then the 64 imaginary parts) x CT_BN = 64
// intermediates m, K walked in chunks of CT_BK = 8 insertion pairs c (16 real k: 8 real parts, then 8 imaginary parts), the
// tiles of two chunks in shared memory (one barrier per chunk: a warp stores the next chunk as soon as ITS DMMAs are done).
// 8 warps as 4 (32 real rows) x 2 (32 columns): 16 accumulator tiles of 8 x 8 per warp, 16 DMMAs per 8 fragment loads.
// Once per CTA the 64 columns get their index terms X[q], Y[l] (mcb_device.cuh) and factors sqrt(m_j + 1), sqrt((m_j+1)(m_j+2))
// in shared memory; a B element is then one gather of C and one or two multiplications.  The next chunk's global loads (Vp
// and the gathers) are issued into registers before the DMMAs of the current chunk.
#define CT_BM 64
#define CT_BN 64
#define CT_BK 8
#define CT_PER (CT_BM * CT_BK / CT_THREADS)   // elements of an A tile (and of a B tile) per thread and chunk
#define CT_THREADS 256
#define CT_LDA (2 * CT_BK + 4)        // doubles; % 16 == 4: conflict-free A fragments
#define CT_LDB (CT_BN + 4)            // doubles; % 16 == 4: conflict-free B fragments

__device__ __forceinline__ void big_dmma884(double& c0, double& c1, const double a, const double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// the DMMAs of one K chunk for the first NB 8-row blocks of the warp (a branch per warp, not a predicate per DMMA: a
// predicated-off DMMA still takes its slot in the tensor pipe)
template <int NB>
__device__ __forceinline__ void ct_chunk(double (&acc)[4][4][2], const double* __restrict__ xa, const double* __restrict__ xb)
{
#pragma unroll
    for (int ks = 0; ks < 2 * CT_BK / 4; ++ks) {
        double a[NB > 0 ? NB : 1], b[4];
#pragma unroll
        for (int i = 0; i < NB; ++i) a[i] = xa[8 * i * CT_LDA + 4 * ks];
#pragma unroll
        for (int j = 0; j < 4; ++j) b[j] = xb[4 * ks * CT_LDB + 8 * j];
#pragma unroll
        for (int i = 0; i < NB; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) big_dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
}

static size_t big_contract_smem(int M)
{
    return sizeof(double) * (2 * ((size_t)2 * CT_BM * CT_LDA + (size_t)2 * CT_BK * CT_LDB) + (size_t)2 * M * CT_BN) + sizeof(int) * (size_t)2 * M * CT_BN;
}

__global__ void __launch_bounds__(CT_THREADS) k_big_contract(const BigArgs p, const unsigned short* __restrict__ pair_k, const unsigned short* __restrict__ pair_s)
{
    extern __shared__ __align__(16) double ct_smem[];
    const McbDev& d = p.d;
    const int M = d.M, P = p.P;
    constexpr int STAGE = 2 * CT_BM * CT_LDA + 2 * CT_BK * CT_LDB;       // doubles per stage: A [2 BM][LDA], then B [2 BK][LDB]
    double* sR1 = ct_smem + 2 * STAGE;                                   // [M][BN] sqrt(m_j + 1)
    double* sR2 = sR1 + M * CT_BN;                                       // [M][BN] sqrt((m_j + 1)(m_j + 2))
    int* sX = reinterpret_cast<int*>(sR2 + M * CT_BN);                   // [M][BN]
    int* sY = sX + M * CT_BN;                                            // [M][BN]
    const int a0 = blockIdx.y * CT_BM, m0 = blockIdx.x * CT_BN;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int grp = lane >> 2, tig = lane & 3;
    const int wr = warp >> 1, wc = warp & 1;

    if (tid < CT_BN) {                                                   // per-column index terms and factors
        const int m = m0 + tid;
        int S[MCB_MAX_M], X[MCB_MAX_M], Y[MCB_MAX_M];
        int run = 0;
        for (int j = 0; j < M; ++j) {
            const int nj = m < d.nc2 ? (int)p.fock.occ2[(long long)j * p.fock.ld2 + m] : 0;
            run += nj; S[j] = run;
            sR1[j * CT_BN + tid] = __ldg(d.sq + nj + 1);
            sR2[j * CT_BN + tid] = __ldg(d.sq2 + nj + 2);
        }
        big_xy(d, S, X, Y);
        for (int j = 0; j < M; ++j) { sX[j * CT_BN + tid] = X[j]; sY[j * CT_BN + tid] = Y[j]; }
    }
    __syncthreads();

    // global -> register staging of one K chunk: 4 elements of Vp and 4 gathered, scaled elements of D per thread
    const int bcol = tid & (CT_BN - 1), bk0 = tid >> 6;                  // B: column, first k of the thread (k = bk0 + 4 i)
    const int ak = tid & (CT_BK - 1), ar0 = tid / CT_BK;                 // A: k within the chunk, first row (row = ar0 + AR i)
    constexpr int AR = CT_THREADS / CT_BK;
    const bool col_ok = m0 + bcol < d.nc2;
    const int base = d.nc - 1;
    double2 ra[CT_PER], rb[CT_PER];
    double rf[CT_PER];                                                   // F(m,c): multiplied in at the stash, AFTER the DMMAs -- the
    auto fetch = [&](int c0) {                                           // gathered value must not be touched while it is in flight
#pragma unroll
        for (int i = 0; i < CT_PER; ++i) {
            const int a = a0 + ar0 + AR * i, c = c0 + ak;
            ra[i] = (a < P && c < P) ? __ldg(p.Vp + (long long)a * P + c) : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int i = 0; i < CT_PER; ++i) {
            const int c = c0 + bk0 + 4 * i;
            rb[i] = make_double2(0.0, 0.0);
            rf[i] = 0.0;
            if (c < P && col_ok) {
                const int q = pair_k[c], l = pair_s[c];
                rb[i] = __ldg(p.C + MCB_CHK(d, base - sX[q * CT_BN + bcol] - sY[l * CT_BN + bcol], d.nc, 203));
                rf[i] = (q == l) ? sR2[q * CT_BN + bcol] : sR1[q * CT_BN + bcol] * sR1[l * CT_BN + bcol];
            }
        }
    };
    auto stash = [&](int stage) {
        double* As = ct_smem + stage * STAGE;
        double* Bs = As + 2 * CT_BM * CT_LDA;
#pragma unroll
        for (int i = 0; i < CT_PER; ++i) {
            const int r = ar0 + AR * i;
            As[r * CT_LDA + ak] = ra[i].x;              As[r * CT_LDA + CT_BK + ak] = -ra[i].y;
            As[(CT_BM + r) * CT_LDA + ak] = ra[i].y;    As[(CT_BM + r) * CT_LDA + CT_BK + ak] = ra[i].x;
        }
#pragma unroll
        for (int i = 0; i < CT_PER; ++i) {
            const int kk = bk0 + 4 * i;
            Bs[kk * CT_LDB + bcol] = rf[i] * rb[i].x;
            Bs[(CT_BK + kk) * CT_LDB + bcol] = rf[i] * rb[i].y;
        }
    };

    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }

    // 8-row blocks of this warp that hold rows a < P (the last row tile is ragged: P = 136 fills 17 of its 24 blocks); the
    // DMMAs of the empty ones are skipped, warp-uniformly
    const int nblk = min(4, max(0, (P - (a0 + 32 * (wr & 1)) + 7) >> 3));
    fetch(0);
    stash(0);
    __syncthreads();
    int stage = 0;
    for (int c0 = 0; c0 < P; c0 += CT_BK, stage ^= 1) {
        const bool more = c0 + CT_BK < P;
        if (more) fetch(c0 + CT_BK);                                     // in flight under the DMMAs below
        const double* xa = ct_smem + stage * STAGE + (32 * wr + grp) * CT_LDA + tig;
        const double* xb = ct_smem + stage * STAGE + 2 * CT_BM * CT_LDA + tig * CT_LDB + 32 * wc + grp;
        switch (nblk) {                                                  // warp-uniform
        case 4: ct_chunk<4>(acc, xa, xb); break;
        case 3: ct_chunk<3>(acc, xa, xb); break;
        case 2: ct_chunk<2>(acc, xa, xb); break;
        case 1: ct_chunk<1>(acc, xa, xb); break;
        default: break;
        }
        // the other stage was last read in the previous iteration, before its closing barrier: free to overwrite now
        if (more) stash(stage ^ 1);
        __syncthreads();
    }

    // epilogue: real row 32 wr + 8 i + grp = (part, a - a0) with part = wr >> 1; columns 32 wc + 8 j + 2 tig, + 1
    const int part = wr >> 1;
    double* Wd = reinterpret_cast<double*>(p.W);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int a = a0 + 32 * (wr & 1) + 8 * i + grp;
        if (a >= P) continue;
        const int k = pair_k[a], s = pair_s[a];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int col = 32 * wc + 8 * j + 2 * tig + e;
                const int m = m0 + col;
                if (m >= d.nc2) continue;
                const double f = (k == s) ? sR2[k * CT_BN + col] : sR1[k * CT_BN + col] * sR1[s * CT_BN + col];
                Wd[2 * ((long long)a * p.ld2 + m) + part] = f * acc[i][j][e];
            }
        }
    }
}

// HC[g] = sum over allowed removal pairs (k<=s) of W'[pair(k,s)][index2(n^g - e_k - e_s)]; one thread per output
__global__ void __launch_bounds__(BIG_THREADS) k_big_reduce(const BigArgs p)
{
    const McbDev& d = p.d;
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= d.nc) return;
    const int M = d.M;
    int n[MCB_MAX_M], X[MCB_MAX_M], Y[MCB_MAX_M];
    {
        int A1[MCB_MAX_M], A2[MCB_MAX_M];
        int run = 0, x = 0, tot1 = 0;
        for (int j = 0; j < M; ++j) {
            n[j] = p.fock.occ[(long long)j * p.fock.ld + g];
            run += n[j];
            X[j] = x;
            if (j <= M - 2) {
                // prefix sums of n - e_k - e_s: S_j (j < k), S_j - 1 (k <= j < s), S_j - 2 (j >= s)
                const int a0 = mcb_ldG(d.G, d.ldg, j, run);
                A1[j] = mcb_ldG(d.G, d.ldg, j, run >= 1 ? run - 1 : 0);
                A2[j] = mcb_ldG(d.G, d.ldg, j, run >= 2 ? run - 2 : 0);
                x += a0 - A1[j]; tot1 += A1[j];
            } else { A1[j] = 0; A2[j] = 0; }
        }
        int pre = tot1, suf = 0;
        for (int l = M - 1; l >= 0; --l) { pre -= A1[l]; suf += A2[l]; Y[l] = pre + suf; }
    }
    double re = 0.0, im = 0.0;
    for (int k = 0; k < M; ++k) {
        if (n[k] < 1) continue;
        for (int s = k; s < M; ++s) {
            if ((k == s) ? (n[k] < 2) : (n[s] < 1)) continue;
            const double2 w = p.W[(long long)mcb_pair_index(M, k, s) * p.ld2 + MCB_CHK(d, d.nc2 - 1 - X[k] - Y[s], d.nc2, 202)];
            re += w.x; im += w.y;
        }
    }
    p.HC[g] = make_double2(re, im);
}

// N = 1: HC = T.C over the M one-particle configurations (Algorithm 1 gives |e_j> the index j)
__global__ void k_big_onebody(const double2* __restrict__ Tm, const double2* __restrict__ C, double2* __restrict__ HC, int M)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= M) return;
    double re = 0.0, im = 0.0;
    for (int l = 0; l < M; ++l) {
        const double2 t = Tm[k * M + l], c = C[l];
        re += t.x * c.x - t.y * c.y; im += t.x * c.y + t.y * c.x;
    }
    HC[k] = make_double2(re, im);
}

// partial[z][a][c] = sum over the m-slice z of conj(D[a][m]) D[c][m]; 32 x 32 tile per CTA, 256 threads, 4 elements each
__global__ void __launch_bounds__(256) k_big_gram(const double2* __restrict__ D, long long ld2, int P, int nc2, int per_split, double2* __restrict__ partial)
{
    __shared__ double2 Ra[32][33], Rc[32][33];
    const int a0 = blockIdx.y * 32, c0 = blockIdx.x * 32;
    const int tid = threadIdx.x, ty = tid >> 5, tx = tid & 31;
    const int mlo = blockIdx.z * per_split, mhi = min(nc2, mlo + per_split);
    double2 acc[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) acc[i] = make_double2(0.0, 0.0);
    for (int m0 = mlo; m0 < mhi; m0 += 32) {
        for (int e = tid; e < 32 * 32; e += 256) {
            const int r = e >> 5, mm = e & 31;
            const bool ok = m0 + mm < mhi;
            Ra[r][mm] = (ok && a0 + r < P) ? D[(long long)(a0 + r) * ld2 + m0 + mm] : make_double2(0.0, 0.0);
            Rc[r][mm] = (ok && c0 + r < P) ? D[(long long)(c0 + r) * ld2 + m0 + mm] : make_double2(0.0, 0.0);
        }
        __syncthreads();
#pragma unroll 8
        for (int mm = 0; mm < 32; ++mm) {
            const double2 c = Rc[tx][mm];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const double2 a = Ra[ty + 8 * i][mm];
                acc[i].x += a.x * c.x + a.y * c.y;
                acc[i].y += a.x * c.y - a.y * c.x;
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int a = a0 + ty + 8 * i, c = c0 + tx;
        if (a < P && c < P) partial[((long long)blockIdx.z * P + a) * P + c] = acc[i];
    }
}

__global__ void k_big_gram_finish(const double2* __restrict__ partial, int nsplit, int P, double2* __restrict__ G)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= P * P) return;
    double re = 0.0, im = 0.0;
    for (int z = 0; z < nsplit; ++z) { const double2 v = partial[(long long)z * P * P + e]; re += v.x; im += v.y; }
    G[e] = make_double2(re, im);
}

// =========================================================================================================
// host
// =========================================================================================================
static long long big_ld2(const mcb_space* sp) { return mcb_round_up(sp->nc2 > 0 ? sp->nc2 : 1, 128); }

long long mcb_big_workspace_bytes(const mcb_space* sp)
{
    // W', P x ld2 complex (the gathered D is never materialised by the apply: k_big_contract)
    return (long long)sp->P * big_ld2(sp) * (long long)sizeof(double2);
}

static int big_pair_tables(mcb_space* sp) { return mcb_pair_tables(sp); }

static void big_args(const mcb_space* sp, const mcb_c128* d_C, mcb_c128* d_HC, void* d_ws, BigArgs& a)
{
    a.d = sp->dev; a.fock = sp->fock;
    a.C = (const double2*)d_C; a.HC = (double2*)d_HC;
    a.Vp = (const double2*)sp->d_coef;
    a.ld2 = big_ld2(sp);
    a.P = sp->P;
    a.D = (double2*)d_ws;
    a.W = a.D + (long long)sp->P * a.ld2;
}

int mcb_launch_big(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_C, mcb_c128* d_HC, void* d_ws, cudaStream_t st)
{
    const int P = sp->P, M = sp->M;
    if (sp->N < 2) {
        // one-body only: HC = T.C (M x M)
        const size_t bytes = sizeof(mcb_c128) * (size_t)M * M;
        if (bytes > sp->coef_bytes) return MCB_ENOMEM;
        if (mcb_coef_stale(sp)) {
            memcpy(sp->h_coef, T, bytes);
            { int rc = mcb_coef_upload(sp, sp->h_coef, bytes, st); if (rc) return rc; }
            mcb_coef_staged(sp);
        }
        { int rc = mcb_tick(sp, 0, st); if (rc) return rc; }
        k_big_onebody<<<(M + 63) / 64, 64, 0, st>>>((const double2*)sp->d_coef, (const double2*)d_C, (double2*)d_HC, M);
        MCB_CHECK_LAUNCH();
        { int rc = mcb_tick(sp, 1, st); if (rc) return rc; }
        mcb_tick_done(sp, 1);
        sp->last_launches = 1;
        return MCB_OK;
    }
    { int rc = big_pair_tables(sp); if (rc) return rc; }
    // Vp (T folded in), interleaved complex, staged through the space's host scratch
    const size_t pp = (size_t)P * P;
    if (sizeof(double) * 4 * pp > sp->coef_bytes) return MCB_ENOMEM;
    if (mcb_coef_stale(sp)) {                                            // (a Lanczos run stages them once: M^4 entries, 1e6 at M = 32)
        double* h = (double*)sp->h_coef;
        double* vr = h + 2 * pp;
        double* vi = vr + pp;
        mcb_pack_pairs(sp->N, M, T, V, true, vr, vi);
        for (size_t i = 0; i < pp; ++i) { h[2 * i] = vr[i]; h[2 * i + 1] = vi[i]; }
        { int rc = mcb_coef_upload(sp, h, sizeof(double) * 2 * pp, st); if (rc) return rc; }
        mcb_coef_staged(sp);
    }
    BigArgs a;
    big_args(sp, d_C, d_HC, d_ws, a);
    a.D = nullptr; a.W = (double2*)d_ws;                                 // the workspace is W' alone
    const size_t smem = big_contract_smem(M);
    if (!(sp->attr_set & (1u << 9))) {
        MCB_CUDA(cudaFuncSetAttribute(k_big_contract, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)big_contract_smem(MCB_MAX_M)));
        sp->attr_set |= 1u << 9;
    }
    { int rc = mcb_tick(sp, 0, st); if (rc) return rc; }
    const dim3 grid((unsigned)((sp->nc2 + CT_BN - 1) / CT_BN), (unsigned)((P + CT_BM - 1) / CT_BM));
    k_big_contract<<<grid, CT_THREADS, smem, st>>>(a, sp->d_pair_ks, sp->d_pair_ks + P);
    MCB_CHECK_LAUNCH();
    { int rc = mcb_tick(sp, 1, st); if (rc) return rc; }
    k_big_reduce<<<(unsigned)((sp->nc + BIG_THREADS - 1) / BIG_THREADS), BIG_THREADS, 0, st>>>(a);
    MCB_CHECK_LAUNCH();
    { int rc = mcb_tick(sp, 2, st); if (rc) return rc; }
    mcb_tick_done(sp, 2);
    sp->last_launches = 2;
    return MCB_OK;
}

// ---- density matrices for M > 12 ------------------------------------------------------------------------------------
static int big_nsplit(const mcb_space* sp)
{
    long long s = (sp->nc2 + 4095) / 4096;                              // at least 4096 intermediates per slice
    if (s < 1) s = 1;
    if (s > BIG_SPLIT_MAX) s = BIG_SPLIT_MAX;
    return (int)s;
}

long long mcb_big_rho_workspace_bytes(const mcb_space* sp)
{
    const long long pp = (long long)sp->P * sp->P * (long long)sizeof(double2);
    return (long long)sp->P * big_ld2(sp) * (long long)sizeof(double2)   // D
           + mcb_round_up((long long)big_nsplit(sp) * pp, 256)          // partial Gram matrices
           + mcb_round_up(pp, 256);                                     // G
}

int mcb_launch_rho_big(mcb_space* sp, const mcb_c128* d_C, mcb_c128* d_rho1, mcb_c128* d_rho2, void* d_ws, cudaStream_t st)
{
    const int P = sp->P, M = sp->M;
    const long long pp = (long long)P * P * (long long)sizeof(double2);
    BigArgs a;
    big_args(sp, d_C, NULL, d_ws, a);
    double2* partial = a.D + (long long)P * a.ld2;
    const int nsplit = big_nsplit(sp);
    double2* G = (double2*)((char*)partial + mcb_round_up((long long)nsplit * pp, 256));
    int launches = 0;
    if (sp->N >= 2) {
        k_big_gather<<<(unsigned)((sp->nc2 + BIG_THREADS - 1) / BIG_THREADS), BIG_THREADS, 0, st>>>(a);
        MCB_CHECK_LAUNCH();
        const int per_split = (int)mcb_round_up((sp->nc2 + nsplit - 1) / nsplit, 32);
        const dim3 grid((unsigned)((P + 31) / 32), (unsigned)((P + 31) / 32), (unsigned)nsplit);
        k_big_gram<<<grid, 256, 0, st>>>(a.D, a.ld2, P, (int)sp->nc2, per_split, partial);
        MCB_CHECK_LAUNCH();
        k_big_gram_finish<<<(P * P + 255) / 256, 256, 0, st>>>(partial, nsplit, P, G);
        MCB_CHECK_LAUNCH();
        launches = 3;
    }
    { int rc = mcb_rho_expand_launch(G, d_C, sp->N, M, d_rho1, d_rho2, st); if (rc) return rc; }
    sp->last_launches = launches + 1;
    return MCB_OK;
}
