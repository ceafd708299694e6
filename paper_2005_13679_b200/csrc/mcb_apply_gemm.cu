// mcb_apply_gemm.cu -- MCB_GEMM mode of hc_apply (Eq. 12-13): the two-body operator factored
// through the (N-2)-particle space,
//     H2 = sum_m sum_{a=(k<=s)} sum_{c=(q<=l)} |m+e_k+e_s> F(m,a) Vp[a][c] F(m,c) <m+e_q+e_l|,
//     F(m,(q,l)) = sqrt((m_q+1)(m_l+1+[q==l])),
// so that per intermediate m the work is a dense P x P complex mat-vec, and batched over m a (P x P).(P x nc2)
// complex GEMM on the FP64 tensor path (mma.sync m8n8k4 f64 -> SASS DMMA).  T rides along inside Vp
// (sum_s a+_s a_s = N).  Two kernels:
//   k_hc2_contract<M>  persistent, warp-specialised: PRODUCER warps compute the target indices of a tile of TM
//                      intermediates from the hashing table (index = nc-1-X[q]-Y[l], mcb_device.cuh), gather C,
//                      scale by F(m,c) and fill a shared-memory stage D[c][m]; CONSUMER warps hold the packed
//                      coefficient matrix as register-stationary DMMA A-fragments, multiply the stage, scale by
//                      F(m,a) and write W'[a][m] (complex, interleaved).  Stages are handed over with mbarriers
//                      (full/empty ring), so the gathers of tile t+1 run under the DMMAs of tile t.
//   k_hc2_reduce<M>    HC[g] = sum over allowed removal pairs a of W'[a][index2(n^g - e_k - e_s)]: every W' element
//                      is read by exactly one g -- no atomics on the output.
#include <string.h>
#include "mcb_device.cuh"

__host__ __device__ constexpr int cmax(int a, int b) { return a > b ? a : b; }
__host__ __device__ constexpr int cdiv(int a, int b) { return (a + b - 1) / b; }

// Tile shape per M (compile time).
//   EMBED (small M): the complex P x P product is embedded as a real 2P x 2P one with rows ordered (a, re|im):
//        row 2a   = [ Vr[a][:] | -Vi[a][:] ],  row 2a+1 = [ Vi[a][:] | Vr[a][:] ],  D rows = [ Dr ; Di ],
//        which pads 2P (not P) to the 8 x 4 fragment grid;
//   otherwise: real fragments of Vr, Vi and three accumulators Vr.Dr, Vi.Di, (Vr + Vi).(Dr + Di): the complex
//        product with three real multiplications (re = t0 - t1, im = t2 - t0 - t1).
// Consumer warp (wr, wc) owns row blocks {wr, wr + WR, ..} (8 rows each) for ALL k-steps and sweeps the column
// blocks (8 intermediates each) {2 wc, 2 wc + 1, 2 wc + 2 WC, ..} of the tile.
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
    // M = 9, 10: two consumer warps per row block (each sweeps half of the column blocks): 14 DMMA-issuing warps per SM instead
    // of 7 keep the FP64 tensor pipe fed (configs[3]: contract 3.67 -> 3.40 ms); at M >= 11 the 80 registers of A-fragments per
    // warp leave no room for that under the 128-register cap of a 512-thread CTA
    static constexpr int WC = (!EMBED && M <= 10) ? 2 : (WR >= 4 ? 1 : (WR >= 2 ? 2 : 4));
    static constexpr int NWC = WR * WC;                     // consumer warps
    // producer warps.  M >= 9: two -- the fewer threads the CTA has, the more registers a consumer warp gets, and with the
    // 128-register cap of a 448-thread CTA the consumers could not keep the next k-step's fragments in flight (measured at
    // configs[4], M = 12: contract 4.43 / 4.13 / 3.61 ms with 6 / 4 / 2 producer warps; configs[3], M = 10: 3.72 / 3.81 / 4.12 / 3.67 ms
    // with 8 / 6 / 4 / 2)
    static constexpr int NWP = EMBED ? 4 : 2;  // producer warps (measured: P = 55 wants 8, P = 78 wants 4)
    static constexpr int NPT = NWP * 32;                    // producer threads
    static constexpr int TM = EMBED ? 128 : 64;             // intermediates per tile
    static constexpr int LD = TM + 4;                       // smem row stride (doubles): LD % 16 == 4 -> conflict-free B frags
    static constexpr int THREADS = (NWC + NWP) * 32;
    static constexpr int NPARTS = NPT / TM;                 // producer threads per intermediate
    static constexpr int DROWS = NK * 4;                    // rows of each staged D plane
    static constexpr int NPLANES = EMBED ? 1 : 2;
    static constexpr int STAGE = NPLANES * DROWS * LD + 2 * M * TM;   // doubles per stage: D planes, R1, R2
    static constexpr int STAGES = 2;
    static constexpr int MINB = (M <= 6) ? 2 : 1;           // CTAs per SM the register budget is shaped for
    static constexpr int GATHER_BATCH = (M >= 11) ? 13 : 8; // C gathers in flight per producer thread
    static constexpr int A_ROWS = RB * 8, A_COLS = NK * 4;  // padded coefficient matrix (row-major), x PER matrices
    static constexpr size_t SMEM = (size_t)STAGES * STAGE * sizeof(double) + 2 * STAGES * sizeof(unsigned long long);
    static_assert(NPT % TM == 0 && NPARTS >= 1, "producer mapping");
    static_assert((TM / 8) % (2 * WC) == 0, "column sweep");
};

struct GemmArgs {
    McbDev d;
    McbFockView fock;
    const double2* C;
    double2* HC;
    const double* A;           // EMBED: [A_ROWS][A_COLS]; else Vr [A_ROWS][A_COLS] then Vi [A_ROWS][A_COLS]
    double2* W;                // [P][ldw]: W'[a][m] = F(m,a) * sum_c Vp[a][c] F(m,c) C[m + e_q + e_l]
    long long ldw;
    int tile0, ntiles;         // contract: tiles [tile0, ntiles) of this launch
    int g0, g1;                // reduce: outputs [g0, g1) of this launch
};

__device__ __forceinline__ void dmma884(double& c0, double& c1, const double a, const double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// ---- mbarrier (shared::cta) ------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    unsigned ok;
    const unsigned addr = smem_u32(bar);
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(addr), "r"(parity) : "memory");
    } while (!ok);
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
__global__ void __launch_bounds__(GemmCfg<M>::THREADS, GemmCfg<M>::MINB) k_hc2_contract(GemmArgs p)
{
    using Cfg = GemmCfg<M>;
    constexpr int P = Cfg::P, NK = Cfg::NK, NRB = Cfg::NRB, WR = Cfg::WR, WC = Cfg::WC, TM = Cfg::TM, LD = Cfg::LD;
    constexpr int STAGES = Cfg::STAGES;
    constexpr bool EMBED = Cfg::EMBED;
    extern __shared__ double smem[];
    unsigned long long* full = reinterpret_cast<unsigned long long*>(smem + STAGES * Cfg::STAGE);
    unsigned long long* empty = full + STAGES;
    const McbDev& d = p.d;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // zero the stages once (the padding rows of the D planes are never written again), init the barriers
    for (int i = tid; i < STAGES * Cfg::STAGE; i += Cfg::THREADS) smem[i] = 0.0;
    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full + s, Cfg::NPT); mbar_init(empty + s, Cfg::NWC * 32); }
    }
    __syncthreads();

    if (warp >= Cfg::NWC) {
        // ================================ PRODUCER: D[c][m] = F(m,c) C[index(m + e_q + e_l)] ====================
        const int ptid = tid - Cfg::NWC * 32;
        const int m_local = ptid % TM;
        const int part = ptid / TM;
        int it = 0;
        // the occupations of the NEXT tile are loaded while this one is gathered: one memory latency less per tile on the
        // producers' critical path (consumers were waiting on full stages 22 % of their time, profiles/r1_cfg4_gemm_v2.md)
        // (not at M >= 11: the 128-register cap of the 448-thread CTA would spill)
        constexpr bool PREF = M <= 10;
        int occ_next[M];
        if (PREF) {
            const int m0 = (p.tile0 + blockIdx.x) * TM + m_local;
#pragma unroll
            for (int j = 0; j < M; ++j) occ_next[j] = (p.tile0 + blockIdx.x < p.ntiles && m0 < d.nc2) ? (int)p.fock.occ2[(long long)j * p.fock.ld2 + m0] : 0;
        }
        for (int tile = p.tile0 + blockIdx.x; tile < p.ntiles; tile += gridDim.x, ++it) {
            const int s = it % STAGES;
            double* Dr = smem + s * Cfg::STAGE;                  // [DROWS][LD]   (EMBED: rows 0..P-1 real, P..2P-1 imag)
            double* Di = Dr + Cfg::DROWS * LD;                   // [DROWS][LD]   (non-EMBED only)
            double* R1 = Dr + Cfg::NPLANES * Cfg::DROWS * LD;    // [M][TM]  sqrt(m_j + 1)
            double* R2 = R1 + M * TM;                            // [M][TM]  sqrt((m_j + 1)(m_j + 2))
            const int m = tile * TM + m_local;
            const bool valid = m < d.nc2;
            int X[M], Y[M];
            double r1[M], r2[M];
            {
                int A1[M], A2[M];
                int run = 0, x = 0, tot1 = 0;
#pragma unroll
                for (int j = 0; j < M; ++j) {
                    const int nj = PREF ? occ_next[j] : (valid ? (int)p.fock.occ2[(long long)j * p.fock.ld2 + m] : 0);
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
            if (PREF) {
                const int tn = tile + gridDim.x;
                const int mn = tn * TM + m_local;
                const bool vn = tn < p.ntiles && mn < d.nc2;
#pragma unroll
                for (int j = 0; j < M; ++j) occ_next[j] = vn ? (int)p.fock.occ2[(long long)j * p.fock.ld2 + mn] : 0;
            }
            // gathers are issued in batches of GB per thread; the first batch is in flight BEFORE the wait for the
            // stage, so its latency hides under the consumers draining the previous use of this stage
            constexpr int NPARTS = Cfg::NPARTS, GB = Cfg::GATHER_BATCH;
            constexpr int NBATCH = cdiv(P, GB * NPARTS);
#pragma unroll
            for (int b = 0; b < NBATCH; ++b) {
                double2 z[GB];
                {
                    int c = 0;                                              // compile-time after unrolling
#pragma unroll
                    for (int q = 0; q < M; ++q) {
#pragma unroll
                        for (int l = q; l < M; ++l, ++c) {
                            if (c / (GB * NPARTS) == b && (NPARTS == 1 || (c % NPARTS) == part)) {
                                const int tgt = d.nc - 1 - X[q] - Y[l];
                                z[(c % (GB * NPARTS)) / NPARTS] = valid ? __ldg(p.C + MCB_CHK(d, tgt, d.nc, 301)) : make_double2(0.0, 0.0);
                            }
                        }
                    }
                }
                if (b == 0) {
                    mbar_wait(empty + s, ((it / STAGES) & 1) ^ 1);
                    if (part == 0) {
#pragma unroll
                        for (int j = 0; j < M; ++j) { R1[j * TM + m_local] = r1[j]; R2[j * TM + m_local] = r2[j]; }
                    }
                }
                {
                    int c = 0;
#pragma unroll
                    for (int q = 0; q < M; ++q) {
#pragma unroll
                        for (int l = q; l < M; ++l, ++c) {
                            if (c / (GB * NPARTS) == b && (NPARTS == 1 || (c % NPARTS) == part)) {
                                const double f = (q == l) ? r2[q] : r1[q] * r1[l];
                                const double2 v = z[(c % (GB * NPARTS)) / NPARTS];
                                if (EMBED) { Dr[c * LD + m_local] = f * v.x; Dr[(P + c) * LD + m_local] = f * v.y; }
                                else       { Dr[c * LD + m_local] = f * v.x; Di[c * LD + m_local] = f * v.y; }
                            }
                        }
                    }
                }
            }
            mbar_arrive(full + s);
        }
        return;
    }

    // ==================================== CONSUMER: W' = F . (A . D) ==========================================
    const int wr = warp % WR, wc = warp / WR;
    const int grp = lane >> 2, tig = lane & 3;
    // stationary A fragments: a[rb][ks] = A[(rbg*8 + grp)][ks*4 + tig]
    double a_re[NRB][NK];
    double a_im[EMBED ? 1 : NRB][EMBED ? 1 : NK];
    int row_k[NRB], row_s[NRB];                               // the removal pair of this lane's accumulator row
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
        const int pr = EMBED ? (r >> 1) : r;
        int k = 0, s = 0;
        const bool row_live = live && pr < P;
        if (row_live) pair_decode(M, pr, k, s);
        row_k[i] = row_live ? k : -1; row_s[i] = s;
    }

    int it = 0;
    for (int tile = p.tile0 + blockIdx.x; tile < p.ntiles; tile += gridDim.x, ++it) {
        const int s = it % STAGES;
        const double* Dr = smem + s * Cfg::STAGE;
        const double* R1 = Dr + Cfg::NPLANES * Cfg::DROWS * LD;
        const double* R2 = R1 + M * TM;
        const int m0 = tile * TM;
        mbar_wait(full + s, (it / STAGES) & 1);
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
                const double bs0 = br0 + bi0, bs1 = br1 + bi1;
#pragma unroll
                for (int i = 0; i < NRB; ++i) {
                    if (EMBED) {
                        dmma884(acc[i][0][0][0], acc[i][0][0][1], a_re[i][ks], br0);
                        dmma884(acc[i][1][0][0], acc[i][1][0][1], a_re[i][ks], br1);
                    } else {
                        // complex product with three real ones: Vr.Dr, Vi.Di, (Vr + Vi).(Dr + Di)   (reading A19)
                        const double a_s = a_re[i][ks] + a_im[i][ks];
                        dmma884(acc[i][0][0][0], acc[i][0][0][1], a_re[i][ks], br0);
                        dmma884(acc[i][1][0][0], acc[i][1][0][1], a_re[i][ks], br1);
                        dmma884(acc[i][0][1][0], acc[i][0][1][1], a_im[i][ks], bi0);
                        dmma884(acc[i][1][1][0], acc[i][1][1][1], a_im[i][ks], bi1);
                        dmma884(acc[i][0][2][0], acc[i][0][2][1], a_s, bs0);
                        dmma884(acc[i][1][2][0], acc[i][1][2][1], a_s, bs1);
                    }
                }
            }
            // epilogue: W'[a][m] = F(m,a) * acc.  This lane holds columns col, col+1 of row (rbg*8 + grp).
#pragma unroll
            for (int i = 0; i < NRB; ++i) {
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const int col = (cb + j) * 8 + tig * 2;
                    if (EMBED) {
                        // rows come in (re, im) pairs on lanes grp, grp^1 (lane ^ 4): even lanes end up with the
                        // complex value of column col, odd lanes with that of column col + 1.  The shuffle is
                        // executed by every lane of the warp (dead rows carry zeros).
                        const bool odd = grp & 1;
                        const double give = odd ? acc[i][j][0][0] : acc[i][j][0][1];
                        const double got = __shfl_xor_sync(0xffffffffu, give, 4);
                        if (row_k[i] < 0) continue;
                        const int k = row_k[i], sI = row_s[i];
                        const int mc = col + (odd ? 1 : 0);
                        const double f = (k == sI) ? R2[k * TM + mc] : R1[k * TM + mc] * R1[sI * TM + mc];
                        const double2 o = odd ? make_double2(f * got, f * acc[i][j][0][1]) : make_double2(f * acc[i][j][0][0], f * got);
                        p.W[(size_t)mcb_pair_index(M, k, sI) * p.ldw + m0 + mc] = o;
                    } else {
                        if (row_k[i] < 0) continue;
                        const int k = row_k[i], sI = row_s[i];
                        double f0, f1;
                        if (k == sI) { f0 = R2[k * TM + col]; f1 = R2[k * TM + col + 1]; }
                        else { f0 = R1[k * TM + col] * R1[sI * TM + col]; f1 = R1[k * TM + col + 1] * R1[sI * TM + col + 1]; }
                        double2* w = p.W + (size_t)mcb_pair_index(M, k, sI) * p.ldw + m0 + col;
                        w[0] = make_double2(f0 * (acc[i][j][0][0] - acc[i][j][1][0]), f0 * ((acc[i][j][2][0] - acc[i][j][0][0]) - acc[i][j][1][0]));
                        w[1] = make_double2(f1 * (acc[i][j][0][1] - acc[i][j][1][1]), f1 * ((acc[i][j][2][1] - acc[i][j][0][1]) - acc[i][j][1][1]));
                    }
                }
            }
        }
        mbar_arrive(empty + s);
    }
}

// HC[g] = sum over allowed removal pairs (k<=s) of W'[ks][index2(n^g - e_k - e_s)].  One thread per output.
// (registers pinned by the launch bounds: a latency-bound gather lives on resident warps -- left to itself ptxas takes 93
// registers at M = 12 and halves them, 1.46 ms at configs[4].  Measured, configs[3] / configs[4]: 256 threads x 3 | 4 CTAs with 16
// loads per batch 0.86 / 0.94 ms; 128 threads x 6 | 8 CTAs with 12 | 8 loads per batch 0.80 / 0.88 ms)
#define RED_T 128
template <int M>
__global__ void __launch_bounds__(RED_T, (M >= 11 ? 8 : 6)) k_hc2_reduce(GemmArgs p)
{
    const McbDev& d = p.d;
    const int g = p.g0 + blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= p.g1) return;
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
    // the allowed W' elements are fetched in batches of RB_ loads that are all in flight before the first add
    // (latency-bound gather: run length of the index order is only ~(N+M-1)/(M-1))
    constexpr int P = M * (M + 1) / 2;
    constexpr int REDUCE_BATCH = M >= 11 ? 8 : 12;
    constexpr int RB_ = P <= REDUCE_BATCH ? P : REDUCE_BATCH;
    double re = 0.0, im = 0.0;
    int mi[P];
    bool ok[P];
    {
        int a = 0;
#pragma unroll
        for (int k = 0; k < M; ++k) {
#pragma unroll
            for (int s = k; s < M; ++s, ++a) {
                ok[a] = (k == s) ? (n[k] >= 2) : (n[k] >= 1 && n[s] >= 1);
                mi[a] = d.nc2 - 1 - X[k] - Y[s];
            }
        }
    }
#pragma unroll
    for (int a0 = 0; a0 < P; a0 += RB_) {
        double2 w[RB_];
#pragma unroll
        for (int i = 0; i < RB_; ++i) {
            const int a = a0 + i;
            w[i] = make_double2(0.0, 0.0);
            if (a < P && ok[a]) w[i] = __ldcs(p.W + (size_t)a * p.ldw + MCB_CHK(d, mi[a], d.nc2, 302));
        }
#pragma unroll
        for (int i = 0; i < RB_; ++i) { re += w[i].x; im += w[i].y; }
    }
    p.HC[g] = make_double2(re, im);
}

// =========================================================================================================
// host
// =========================================================================================================
#define MCB_DISPATCH_GEMM_M(M, CALL)                                                                     \
    switch (M) {                                                                                         \
    case 1:  { constexpr int MT = 1;  CALL; } break;  case 2:  { constexpr int MT = 2;  CALL; } break;   \
    case 3:  { constexpr int MT = 3;  CALL; } break;  case 4:  { constexpr int MT = 4;  CALL; } break;   \
    case 5:  { constexpr int MT = 5;  CALL; } break;  case 6:  { constexpr int MT = 6;  CALL; } break;   \
    case 7:  { constexpr int MT = 7;  CALL; } break;  case 8:  { constexpr int MT = 8;  CALL; } break;   \
    case 9:  { constexpr int MT = 9;  CALL; } break;  case 10: { constexpr int MT = 10; CALL; } break;   \
    case 11: { constexpr int MT = 11; CALL; } break;  case 12: { constexpr int MT = 12; CALL; } break;   \
    default: return MCB_EUNSUPPORTED;                                                                    \
    }

static long long gemm_ldw(const mcb_space* sp) { return mcb_round_up(sp->nc2, 128); }

long long mcb_gemm_workspace_bytes(const mcb_space* sp)
{
    return (long long)sp->P * gemm_ldw(sp) * (long long)sizeof(double2);
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
    if (mcb_coef_stale(sp)) {
        mcb_pack_pairs(sp->N, M, T, V, true, vr, vi);
        memset(h, 0, a_bytes);
        for (int a = 0; a < P; ++a)
            for (int c = 0; c < P; ++c) {
                const double re = vr[a * P + c], im = vi[a * P + c];
                if (Cfg::EMBED) {
                    h[(size_t)(2 * a) * Cfg::A_COLS + c] = re;          h[(size_t)(2 * a) * Cfg::A_COLS + P + c] = -im;
                    h[(size_t)(2 * a + 1) * Cfg::A_COLS + c] = im;      h[(size_t)(2 * a + 1) * Cfg::A_COLS + P + c] = re;
                } else {
                    h[(size_t)a * Cfg::A_COLS + c] = re;
                    h[mat + (size_t)a * Cfg::A_COLS + c] = im;
                }
            }
        { int rc = mcb_coef_upload(sp, h, a_bytes, st); if (rc) return rc; }
        mcb_coef_staged(sp);
    }

    GemmArgs g;
    g.d = sp->dev; g.fock = sp->fock;
    g.C = (const double2*)d_C; g.HC = (double2*)d_HC;
    g.A = (const double*)sp->d_coef;
    g.W = (double2*)d_ws; g.ldw = gemm_ldw(sp);
    g.ntiles = (int)((sp->nc2 + Cfg::TM - 1) / Cfg::TM);

    if (!sp->gemm_sms) {                                                 // cached per space (one device, one M)
        int sm_count = 0, ctas_per_sm = 0;
        MCB_CUDA(cudaFuncSetAttribute(k_hc2_contract<M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM));
        MCB_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas_per_sm, k_hc2_contract<M>, Cfg::THREADS, Cfg::SMEM));
        MCB_CUDA(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, sp->device));
        if (ctas_per_sm < 1) return MCB_EUNSUPPORTED;
        sp->gemm_sms = sm_count; sp->gemm_ctas_per_sm = ctas_per_sm;
    }
    const int threads = RED_T;
    if (sp->slabs) {
        // pipelined host apply: per slab (cut by the occupation of the last orbital) the contraction of its intermediates, then
        // the gather of its outputs -- a removal never raises that occupation, so slab k of HC only needs slabs <= k of W'
        long long g0 = 0, m0 = 0;
        int launches = 0;
        for (int k = 0; k < sp->slabs->n; ++k) {
            const long long g1 = sp->slabs->g_end[k], m1 = sp->slabs->m_end[k];
            MCB_CUDA(cudaStreamWaitEvent(st, sp->slabs->ev_in[k], 0));
            if (m1 > m0) {
                g.tile0 = (int)(m0 / Cfg::TM); g.ntiles = (int)((m1 + Cfg::TM - 1) / Cfg::TM);
                int grid = sp->gemm_sms * sp->gemm_ctas_per_sm;
                if (grid > g.ntiles - g.tile0) grid = g.ntiles - g.tile0;
                k_hc2_contract<M><<<grid, Cfg::THREADS, Cfg::SMEM, st>>>(g);
                MCB_CHECK_LAUNCH();
                ++launches;
            }
            if (g1 > g0) {
                g.g0 = (int)g0; g.g1 = (int)g1;
                k_hc2_reduce<M><<<(unsigned)((g1 - g0 + threads - 1) / threads), threads, 0, st>>>(g);
                MCB_CHECK_LAUNCH();
                ++launches;
            }
            MCB_CUDA(cudaEventRecord(sp->slabs->ev_out[k], st));
            g0 = g1; m0 = m1;
        }
        sp->last_launches = launches;
        return MCB_OK;
    }
    g.tile0 = 0; g.g0 = 0; g.g1 = (int)sp->nc;
    int grid = sp->gemm_sms * sp->gemm_ctas_per_sm;
    if (grid > g.ntiles) grid = g.ntiles;
    { int rc = mcb_tick(sp, 0, st); if (rc) return rc; }
    k_hc2_contract<M><<<grid, Cfg::THREADS, Cfg::SMEM, st>>>(g);
    MCB_CHECK_LAUNCH();
    { int rc = mcb_tick(sp, 1, st); if (rc) return rc; }
    k_hc2_reduce<M><<<(unsigned)((sp->nc + threads - 1) / threads), threads, 0, st>>>(g);
    MCB_CHECK_LAUNCH();
    { int rc = mcb_tick(sp, 2, st); if (rc) return rc; }
    mcb_tick_done(sp, 2);
    sp->last_launches = 2;
    return MCB_OK;
}

int mcb_launch_gemm(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_C, mcb_c128* d_HC,
                    void* d_ws, cudaStream_t st)
{
    MCB_DISPATCH_GEMM_M(sp->M, return launch_gemm<MT>(sp, T, V, d_C, d_HC, d_ws, st));
    return MCB_EINVAL;
}
