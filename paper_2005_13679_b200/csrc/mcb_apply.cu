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
#include <string.h>
#include "mcb_device.cuh"

// measurement support (mcb_timing_enable): event i of the current apply's slot, recorded on the apply's stream
static inline int mcb_tick(mcb_space* sp, int i, cudaStream_t st)
{
    if (!sp->timing || sp->t_count >= MCB_TIMING_RING) return MCB_OK;
    MCB_CUDA(cudaEventRecord(sp->t_ev[sp->t_count][i], st));
    return MCB_OK;
}
static inline void mcb_tick_done(mcb_space* sp, int launches)
{
    if (!sp->timing || sp->t_count >= MCB_TIMING_RING) return;
    sp->t_launches[sp->t_count++] = launches;
}

// =========================================================================================================
// host: packing of T, V
// =========================================================================================================

// Vp[a][c], a = pair(k<=s), c = pair(q<=l):  1/2 * sum over the DISTINCT orderings (k',s') of {k,s} and (q',l')
// of {q,l} of Veff[k'][s'][q'][l'].  The bosonic operator a+_k a+_s a_q a_l is symmetric under k<->s and q<->l,
// so the ordered sum of Eq. (13) equals the sum over unordered pairs of Vp times the operator (reading A8).
// With fold_T, Veff = V + (2/(N-1)) T[k][l] delta_sq, which adds sum_kl T_kl a+_k (N^ ) a_l / (N-1) = the one-body
// term on N-particle states.
static void pack_pairs(int N, int M, const mcb_c128* T, const mcb_c128* V, bool fold_T, double* vr, double* vi /* [P][P] */)
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

    // ---- one-body: sum_kl T_kl sqrt(n_k (n_l + 1)) C[g_k^l], diagonal n_k C[g]  (App. B rho_kl, rho_kk) ----
    {
        int PM[M], PP[M];
        if (!USE_MAPS) {
            int pm = 0, pp = 0;
#pragma unroll
            for (int j = 0; j < M; ++j) {
                PM[j] = pm; PP[j] = pp;
                if (j <= M - 2) {
                    int g0 = mcb_ldG(d.G, d.ldg, j, S[j]);
                    int gm = mcb_ldG(d.G, d.ldg, j, S[j] > 0 ? S[j] - 1 : 0);
                    int gp = mcb_ldG(d.G, d.ldg, j, S[j] < d.N ? S[j] + 1 : d.N);
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
                        if (USE_MAPS) tgt = __ldg(p.map1 + (long long)(k * M + l) * p.ld1 + g);
                        else tgt = (k < l) ? g + (PM[l] - PM[k]) : g - (PP[k] - PP[l]);
                        const double2 c = __ldg(p.C + tgt);
                        const double f = rk[k] * rl[l];
                        cfma(acc, t, make_double2(f * c.x, f * c.y));
                    }
                }
            }
        }
    }

    // ---- two-body: sum over allowed removal pairs (k<=s), then all insertion pairs (q<=l) ----
    if (d.N >= 2) {
        int a = 0;
        for (int k = 0; k < M; ++k) {
            for (int s = k; s < M; ++s, ++a) {
                int nk = 0, ns = 0;
#pragma unroll
                for (int j = 0; j < M; ++j) { nk = (j == k) ? n[j] : nk; ns = (j == s) ? n[j] : ns; }
                const bool ok = (k == s) ? (nk >= 2) : (nk >= 1 && ns >= 1);
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
                            const int a0 = mcb_ldG(d.G, d.ldg, j, sp);
                            A1[j] = mcb_ldG(d.G, d.ldg, j, sp + 1);
                            A2[j] = mcb_ldG(d.G, d.ldg, j, sp + 2);
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
                        const int tgt = USE_MAPS ? __ldg(m2 + (long long)c * p.ld2) : d.nc - 1 - X[q] - Y[l];
                        const double2 z = __ldg(p.C + tgt);
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
// MCB_GEMM path
// =========================================================================================================
// Tile shape per M (compile time).  The packed coefficient matrix A is STATIONARY IN REGISTERS as DMMA
// m8n8k4 A-fragments: warp (wr, wc) of a CTA owns row blocks {wr, wr + WR, ..} (8 rows each) for ALL k-steps and
// sweeps the column blocks (8 intermediates m each) {wc, wc + WC, ..} of the CTA's tile of TM intermediates.
//   EMBED (small M): the complex P x P product is embedded as a real 2P x 2P one,
//        [Wr; Wi] = [[Vr, -Vi], [Vi, Vr]] . [Dr; Di], which pads 2P (not P) to the 8 x 4 fragment grid;
//   otherwise: real fragments of Vr, Vi and three accumulators (Vr.Dr, Vi.Di, Vr.Di + Vi.Dr).
constexpr int cmax(int a, int b) { return a > b ? a : b; }
constexpr int cdiv(int a, int b) { return (a + b - 1) / b; }

template <int M> struct GemmCfg {
    static constexpr int P = M * (M + 1) / 2;
    static constexpr bool EMBED = (M <= 8);
    static constexpr int ROWS = EMBED ? 2 * P : P;          // output rows of the real GEMM(s)
    static constexpr int RB = cdiv(ROWS, 8);                // 8-row blocks
    static constexpr int KD = EMBED ? 2 * P : P;            // contraction length
    static constexpr int NK = cdiv(KD, 4);                  // k-steps of 4
    static constexpr int PER = EMBED ? 1 : 2;               // A doubles per (row block, k-step, lane)
    static constexpr int NRB_MAX = cmax(1, 48 / (NK * PER));
    static constexpr int WR = cdiv(RB, NRB_MAX);
    static constexpr int NRB = cdiv(RB, WR);
    static constexpr int WC = WR >= 4 ? 1 : (WR >= 2 ? 2 : 4);
    static constexpr int TM = 128;                          // intermediates per tile
    static constexpr int LD = TM + 4;                       // smem row stride (doubles): LD % 16 == 4 -> conflict-free B frags
    static constexpr int THREADS = WR * WC * 32;
    static constexpr int NPARTS = cmax(1, THREADS / TM);    // gather: threads per intermediate
    static constexpr int DROWS = NK * 4;                    // rows of each staged D plane
    static constexpr int NPLANES = EMBED ? 1 : 2;
    static constexpr int A_ROWS = RB * 8, A_COLS = NK * 4;  // padded coefficient matrix (row-major), x PER matrices
    static constexpr size_t SMEM = (size_t)(NPLANES * DROWS * LD + 2 * M * TM) * sizeof(double);
    static_assert(THREADS >= TM || TM % THREADS == 0, "gather mapping");
};

struct GemmArgs {
    McbDev d;
    McbFockView fock;
    const double2* C;
    double2* HC;
    const double* A;           // EMBED: [A_ROWS][A_COLS]; else Vr [A_ROWS][A_COLS] then Vi [A_ROWS][A_COLS]
    double* W;                 // [P][2][ldw]: W'[ks][re|im][m] = F(m,ks) * sum_ql Vp[ks][ql] F(m,ql) C[m + e_q + e_l]
    long long ldw;
    int ntiles;
};

__device__ __forceinline__ void dmma884(double& c0, double& c1, const double a, const double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// pair index -> (k, s), k <= s, order (0,0),(0,1),..
__device__ __forceinline__ void pair_decode(int M, int a, int& k, int& s)
{
    k = 0;
    int len = M;
    while (a >= len) { a -= len; --len; ++k; }
    s = k + a;
}

template <int M>
__global__ void __launch_bounds__(GemmCfg<M>::THREADS, 1) k_hc2_contract(GemmArgs p)
{
    using Cfg = GemmCfg<M>;
    constexpr int P = Cfg::P, NK = Cfg::NK, NRB = Cfg::NRB, WR = Cfg::WR, WC = Cfg::WC, TM = Cfg::TM, LD = Cfg::LD;
    constexpr bool EMBED = Cfg::EMBED;
    extern __shared__ double smem[];
    double* Dr = smem;                                       // [DROWS][LD]   (EMBED: rows 0..P-1 real, P..2P-1 imag)
    double* Di = smem + Cfg::DROWS * LD;                     // [DROWS][LD]   (non-EMBED only)
    double* R1 = smem + Cfg::NPLANES * Cfg::DROWS * LD;      // [M][TM]  sqrt(m_j + 1)
    double* R2 = R1 + M * TM;                                // [M][TM]  sqrt((m_j + 1)(m_j + 2))
    const McbDev& d = p.d;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wr = warp % WR, wc = warp / WR;
    const int grp = lane >> 2, tig = lane & 3;

    // ---- stationary A fragments: a[rb][ks] = A[(rbg*8 + grp)][ks*4 + tig] ----
    double a_re[NRB][NK];
    double a_im[EMBED ? 1 : NRB][EMBED ? 1 : NK];
    int row_k[NRB], row_s[NRB], row_part[NRB];               // which W' row this lane's accumulator rows are
#pragma unroll
    for (int i = 0; i < NRB; ++i) {
        const int rbg = wr + i * WR;
        const int r = rbg * 8 + grp;
        const bool live = rbg < Cfg::RB;
#pragma unroll
        for (int ks = 0; ks < NK; ++ks) {
            a_re[i][ks] = live ? p.A[(size_t)r * Cfg::A_COLS + ks * 4 + tig] : 0.0;
            if (!EMBED) a_im[i][ks] = live ? p.A[(size_t)(Cfg::A_ROWS + r) * Cfg::A_COLS + ks * 4 + tig] : 0.0;
        }
        int pr = -1, part = 0;
        if (live && r < Cfg::ROWS) { pr = EMBED ? (r % P) : r; part = EMBED ? (r / P) : 0; }
        int k = 0, s = 0;
        if (pr >= 0) pair_decode(M, pr, k, s);
        row_k[i] = pr >= 0 ? k : -1; row_s[i] = s; row_part[i] = part;
    }
    // zero the padding rows of the staged planes once (never written again)
    for (int i = tid; i < Cfg::NPLANES * Cfg::DROWS * LD; i += Cfg::THREADS) smem[i] = 0.0;
    __syncthreads();

    const int m_local = tid % TM;
    const int part = tid / TM;

    for (int tile = blockIdx.x; tile < p.ntiles; tile += gridDim.x) {
        const int m0 = tile * TM;
        // ================= gather: D[ql][m] = F(m,ql) C[index(m + e_q + e_l)] =================
        if (part < Cfg::NPARTS) {
            const int m = m0 + m_local;
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
            if (part == 0) {
#pragma unroll
                for (int j = 0; j < M; ++j) { R1[j * TM + m_local] = r1[j]; R2[j * TM + m_local] = r2[j]; }
            }
            int c = 0;
#pragma unroll
            for (int q = 0; q < M; ++q) {
#pragma unroll
                for (int l = q; l < M; ++l, ++c) {
                    if (Cfg::NPARTS == 1 || (c % Cfg::NPARTS) == part) {
                        const int tgt = d.nc - 1 - X[q] - Y[l];
                        double2 z = make_double2(0.0, 0.0);
                        if (valid) z = __ldg(p.C + tgt);
                        const double f = (q == l) ? r2[q] : r1[q] * r1[l];
                        if (EMBED) { Dr[c * LD + m_local] = f * z.x; Dr[(P + c) * LD + m_local] = f * z.y; }
                        else       { Dr[c * LD + m_local] = f * z.x; Di[c * LD + m_local] = f * z.y; }
                    }
                }
            }
        }
        __syncthreads();

        // ================= contraction on the FP64 tensor cores + scaled store =================
        for (int cb = wc * 2; cb < TM / 8; cb += WC * 2) {
            double acc[NRB][2][EMBED ? 1 : 3][2];
#pragma unroll
            for (int i = 0; i < NRB; ++i)
#pragma unroll
                for (int j = 0; j < 2; ++j)
#pragma unroll
                    for (int t = 0; t < (EMBED ? 1 : 3); ++t) { acc[i][j][t][0] = 0.0; acc[i][j][t][1] = 0.0; }
            const double* b_base = Dr + tig * LD + cb * 8 + grp;
#pragma unroll
            for (int ks = 0; ks < NK; ++ks) {
                const double br0 = b_base[ks * 4 * LD], br1 = b_base[ks * 4 * LD + 8];
                double bi0 = 0.0, bi1 = 0.0;
                if (!EMBED) { bi0 = b_base[Cfg::DROWS * LD + ks * 4 * LD]; bi1 = b_base[Cfg::DROWS * LD + ks * 4 * LD + 8]; }
#pragma unroll
                for (int i = 0; i < NRB; ++i) {
                    if (EMBED) {
                        dmma884(acc[i][0][0][0], acc[i][0][0][1], a_re[i][ks], br0);
                        dmma884(acc[i][1][0][0], acc[i][1][0][1], a_re[i][ks], br1);
                    } else {
                        dmma884(acc[i][0][0][0], acc[i][0][0][1], a_re[i][ks], br0);
                        dmma884(acc[i][1][0][0], acc[i][1][0][1], a_re[i][ks], br1);
                        dmma884(acc[i][0][1][0], acc[i][0][1][1], a_im[i][ks], bi0);
                        dmma884(acc[i][1][1][0], acc[i][1][1][1], a_im[i][ks], bi1);
                        dmma884(acc[i][0][2][0], acc[i][0][2][1], a_re[i][ks], bi0);
                        dmma884(acc[i][1][2][0], acc[i][1][2][1], a_re[i][ks], bi1);
                        dmma884(acc[i][0][2][0], acc[i][0][2][1], a_im[i][ks], br0);
                        dmma884(acc[i][1][2][0], acc[i][1][2][1], a_im[i][ks], br1);
                    }
                }
            }
            // epilogue: W'[ks][part][m] = F(m,ks) * acc;  this lane holds columns col, col+1 of row (rbg*8 + grp)
#pragma unroll
            for (int i = 0; i < NRB; ++i) {
                if (row_k[i] < 0) continue;
                const int k = row_k[i], s = row_s[i];
                const int pr = mcb_pair_index(M, k, s);
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const int col = (cb + j) * 8 + tig * 2;
                    double f0, f1;
                    if (k == s) { f0 = R2[k * TM + col]; f1 = R2[k * TM + col + 1]; }
                    else { f0 = R1[k * TM + col] * R1[s * TM + col]; f1 = R1[k * TM + col + 1] * R1[s * TM + col + 1]; }
                    if (EMBED) {
                        double2 o = make_double2(f0 * acc[i][j][0][0], f1 * acc[i][j][0][1]);
                        *reinterpret_cast<double2*>(p.W + ((size_t)pr * 2 + row_part[i]) * p.ldw + m0 + col) = o;
                    } else {
                        double2 ore = make_double2(f0 * (acc[i][j][0][0] - acc[i][j][1][0]), f1 * (acc[i][j][0][1] - acc[i][j][1][1]));
                        double2 oim = make_double2(f0 * acc[i][j][2][0], f1 * acc[i][j][2][1]);
                        *reinterpret_cast<double2*>(p.W + ((size_t)pr * 2 + 0) * p.ldw + m0 + col) = ore;
                        *reinterpret_cast<double2*>(p.W + ((size_t)pr * 2 + 1) * p.ldw + m0 + col) = oim;
                    }
                }
            }
        }
        __syncthreads();               // the next tile's gather overwrites D, R1, R2
    }
}

// HC[g] = sum over allowed removal pairs (k<=s) of W'[ks][index2(n^g - e_k - e_s)]: every W' element is read by
// exactly one g, so there are no atomics on the output.  One thread per output configuration.
template <int M>
__global__ void __launch_bounds__(256) k_hc2_reduce(GemmArgs p)
{
    const McbDev& d = p.d;
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= d.nc) return;
    int n[M], X[M], Y[M];
    {
        int A1[M], A2[M];
        int run = 0, x = 0, tot1 = 0;
#pragma unroll
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
#pragma unroll
        for (int l = M - 1; l >= 0; --l) { pre -= A1[l]; suf += A2[l]; Y[l] = pre + suf; }
    }
    double re = 0.0, im = 0.0;
    int a = 0;
#pragma unroll
    for (int k = 0; k < M; ++k) {
#pragma unroll
        for (int s = k; s < M; ++s, ++a) {
            const bool ok = (k == s) ? (n[k] >= 2) : (n[k] >= 1 && n[s] >= 1);
            if (ok) {
                const int mi = d.nc2 - 1 - X[k] - Y[s];
                const double* w = p.W + (size_t)a * 2 * p.ldw + mi;
                re += __ldg(w);
                im += __ldg(w + p.ldw);
            }
        }
    }
    p.HC[g] = make_double2(re, im);
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
    if (mode == MCB_AUTO) return sp->N >= 2 ? MCB_GEMM : MCB_REHASH;
    if (mode == MCB_GEMM && sp->N < 2) return MCB_REHASH;     // no (N-2)-particle space: H is one-body only
    return mode;
}

static long long gemm_ldw(const mcb_space* sp) { return mcb_round_up(sp->nc2, 128); }

extern "C" long long mcb_apply_workspace_bytes(const mcb_space* sp, int mode)
{
    if (!sp) return MCB_EINVAL;
    if (sp->M > MCB_MAX_M_APPLY) return MCB_EUNSUPPORTED;
    if (mode < MCB_AUTO || mode > MCB_GEMM) return MCB_EINVAL;
    mode = resolve_mode(sp, mode);
    if (mode != MCB_GEMM) return 0;
    return (long long)sp->P * 2 * gemm_ldw(sp) * (long long)sizeof(double);
}

template <int M>
static int launch_direct(mcb_space* sp, bool use_maps, const mcb_c128* T, const mcb_c128* V,
                         const mcb_c128* d_C, mcb_c128* d_HC, cudaStream_t st)
{
    constexpr int P = M * (M + 1) / 2;
    // coefficients: T [M*M] complex, Vp [P*P] complex (interleaved)
    double* h = (double*)sp->h_coef;
    memcpy(h, T, sizeof(mcb_c128) * M * M);
    {
        double* vr = h + 2 * (M * M + P * P);               // scratch behind the packed block
        double* vi = vr + P * P;
        pack_pairs(sp->N, M, T, V, false, vr, vi);
        for (int i = 0; i < P * P; ++i) { h[2 * (M * M + i)] = vr[i]; h[2 * (M * M + i) + 1] = vi[i]; }
    }
    const size_t bytes = sizeof(mcb_c128) * (size_t)(M * M + P * P);
    MCB_CUDA(cudaMemcpyAsync(sp->d_coef, h, bytes, cudaMemcpyHostToDevice, st));
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

template <int M>
static int launch_gemm(mcb_space* sp, const mcb_c128* T, const mcb_c128* V,
                       const mcb_c128* d_C, mcb_c128* d_HC, void* d_ws, cudaStream_t st)
{
    using Cfg = GemmCfg<M>;
    constexpr int P = Cfg::P;
    // ---- coefficient matrix in the padded fragment grid ----
    double* h = (double*)sp->h_coef;
    const size_t mat = (size_t)Cfg::A_ROWS * Cfg::A_COLS;
    const size_t a_bytes = sizeof(double) * mat * Cfg::PER;
    double* vr = h + mat * Cfg::PER;
    double* vi = vr + P * P;
    if ((char*)(vi + P * P) > (char*)sp->h_coef + sp->coef_bytes) return MCB_ENOMEM;
    pack_pairs(sp->N, M, T, V, true, vr, vi);
    memset(h, 0, a_bytes);
    for (int a = 0; a < P; ++a)
        for (int c = 0; c < P; ++c) {
            const double re = vr[a * P + c], im = vi[a * P + c];
            if (Cfg::EMBED) {
                h[(size_t)a * Cfg::A_COLS + c] = re;            h[(size_t)a * Cfg::A_COLS + P + c] = -im;
                h[(size_t)(P + a) * Cfg::A_COLS + c] = im;      h[(size_t)(P + a) * Cfg::A_COLS + P + c] = re;
            } else {
                h[(size_t)a * Cfg::A_COLS + c] = re;
                h[mat + (size_t)a * Cfg::A_COLS + c] = im;
            }
        }
    MCB_CUDA(cudaMemcpyAsync(sp->d_coef, h, a_bytes, cudaMemcpyHostToDevice, st));

    GemmArgs g;
    g.d = sp->dev; g.fock = sp->fock;
    g.C = (const double2*)d_C; g.HC = (double2*)d_HC;
    g.A = (const double*)sp->d_coef;
    g.W = (double*)d_ws; g.ldw = gemm_ldw(sp);
    g.ntiles = (int)((sp->nc2 + Cfg::TM - 1) / Cfg::TM);

    static int sm_count = 0, ctas_per_sm = 0;
    if (!sm_count) {
        MCB_CUDA(cudaFuncSetAttribute(k_hc2_contract<M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM));
        MCB_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas_per_sm, k_hc2_contract<M>, Cfg::THREADS, Cfg::SMEM));
        MCB_CUDA(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, sp->device));
        if (ctas_per_sm < 1) return MCB_EUNSUPPORTED;
    }
    int grid = sm_count * ctas_per_sm;
    if (grid > g.ntiles) grid = g.ntiles;
    { int rc = mcb_tick(sp, 0, st); if (rc) return rc; }
    k_hc2_contract<M><<<grid, Cfg::THREADS, Cfg::SMEM, st>>>(g);
    MCB_CHECK_LAUNCH();
    { int rc = mcb_tick(sp, 1, st); if (rc) return rc; }
    const int threads = 256;
    k_hc2_reduce<M><<<(unsigned)((sp->nc + threads - 1) / threads), threads, 0, st>>>(g);
    MCB_CHECK_LAUNCH();
    { int rc = mcb_tick(sp, 2, st); if (rc) return rc; }
    mcb_tick_done(sp, 2);
    sp->last_launches = 2;
    return MCB_OK;
}

extern "C" int mcb_hc_apply(mcb_space* sp, const mcb_c128* T, const mcb_c128* V,
                            const mcb_c128* d_C, mcb_c128* d_HC, int mode, void* d_workspace, void* stream)
{
    if (!sp || !T || !V || !d_C || !d_HC) return MCB_EINVAL;
    if (mode < MCB_AUTO || mode > MCB_GEMM) return MCB_EINVAL;
    if (sp->M > MCB_MAX_M_APPLY) return MCB_EUNSUPPORTED;
    if ((((uintptr_t)d_C) & 15) || (((uintptr_t)d_HC) & 15)) return MCB_EINVAL;
    {
        const char* c0 = (const char*)d_C; const char* h0 = (const char*)d_HC;
        const size_t len = (size_t)sp->nc * sizeof(mcb_c128);
        if (c0 < h0 + len && h0 < c0 + len) return MCB_EINVAL;          // overlap
    }
    if (!sp->d_fock) return MCB_ENOTREADY;
    mode = resolve_mode(sp, mode);
    cudaStream_t st = (cudaStream_t)stream;
    if (mode == MCB_MAPS && (!sp->d_map1 || (sp->N >= 2 && !sp->d_map2))) return MCB_ENOTREADY;
    if (mode == MCB_GEMM) {
        if (!d_workspace || (((uintptr_t)d_workspace) & 255)) return MCB_EINVAL;
        MCB_DISPATCH_APPLY_M(sp->M, return launch_gemm<MT>(sp, T, V, d_C, d_HC, d_workspace, st));
    } else {
        const bool use_maps = mode == MCB_MAPS;
        MCB_DISPATCH_APPLY_M(sp->M, return launch_direct<MT>(sp, use_maps, T, V, d_C, d_HC, st));
    }
    return MCB_EINVAL;
}

extern "C" int mcb_hc_apply_host(mcb_space* sp, const mcb_c128* T, const mcb_c128* V,
                                 const mcb_c128* h_C, mcb_c128* h_HC, int mode,
                                 mcb_c128* d_C_scratch, mcb_c128* d_HC_scratch, void* d_workspace, void* stream)
{
    if (!sp || !h_C || !h_HC || !d_C_scratch || !d_HC_scratch) return MCB_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t len = (size_t)sp->nc * sizeof(mcb_c128);
    MCB_CUDA(cudaMemcpyAsync(d_C_scratch, h_C, len, cudaMemcpyHostToDevice, st));
    int rc = mcb_hc_apply(sp, T, V, d_C_scratch, d_HC_scratch, mode, d_workspace, stream);
    if (rc != MCB_OK) return rc;
    MCB_CUDA(cudaMemcpyAsync(h_HC, d_HC_scratch, len, cudaMemcpyDeviceToHost, st));
    MCB_CUDA(cudaStreamSynchronize(st));
    return MCB_OK;
}
