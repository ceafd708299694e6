// mcb_lanczos.cu -- Lanczos tridiagonalisation of H with full re-orthogonalisation, device resident
// ("Lanczos tridiagonal decomposition ... with full re-orthogonalisation", the consumer of H.C in
// the paper's ground-state program), and the host tridiagonal eigen-solve that finishes it
// (the paper hands the tridiagonal problem to LAPACK on the host; here: Sturm bisection, no LAPACK).
//
//   v_0 = v0 / |v0|;   for j = 0 .. k-1:   w = H v_j                                   (mcb_hc_apply, any mode)
//                                          c_i = <v_i|w>, i <= j;  alpha_j = Re c_j    (k_lz_dots + k_lz_finish)
//                                          w -= sum_{i<=j} c_i v_i   (twice: classical Gram-Schmidt, re-orthogonalised)
//                                          beta_j = |w|;  stop if beta_j <= breakdown * max(1, |alpha_0|);  v_{j+1} = w / beta_j
// Orthogonalising against ALL previous vectors removes alpha_j v_j and beta_{j-1} v_{j-1} of the three-term
// recurrence together with the rounding-induced components along older vectors.
//
// Everything of a step stays on the device: alpha, beta, 1/beta and the breakdown flag live in a small state block that
// the kernels read and write themselves, so a step is a fixed sequence of launches with NO host round trip; the host
// looks at the state every LZ_SYNC_EVERY steps (to stop early after a breakdown) and once at the end.
//   k_lz_dots     one pass over w per group of 8 basis vectors: w[g] is read once and multiplied into 8 accumulators
//                 (16 nc (nv + nv/8) bytes instead of the 32 nc nv of a dot product per vector);
//   k_lz_project  w -= sum c_i v_i, and in the same pass the partial sums of |w_new|^2 (the norm costs no extra pass);
//   k_lz_finish   fixed-order sums of the per-block partials: coefficients, alpha, beta, 1/beta, breakdown test.
// All reductions are two-stage with a fixed order (no atomics): the run is bit-reproducible.
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include "mcb_internal.cuh"

#define LZ_THREADS 256
#define LZ_BLOCKS 592                 // partial sums per dot product (4 per SM on a B200)
#define LZ_MAXK 1024
#define LZ_GROUP 8                    // basis vectors per pass over w
#define LZ_SYNC_EVERY 8

struct LzState {                      // device resident
    double alpha[LZ_MAXK];
    double beta[LZ_MAXK];
    double scale;                     // 1 / beta_j (1 / |v0| before the first step): what the next k_lz_scale multiplies by
    double alpha0_abs;
    int k_done;                       // steps completed
    int stop;                         // breakdown (or v0 = 0): every later kernel of the sequence is a no-op
};

// partial[blockIdx.x][i0 + t] = sum over the block's elements of conj(V_{i0+t}[g]) w[g], t < min(LZ_GROUP, nv - i0), i0 = 8 blockIdx.y
__global__ void __launch_bounds__(LZ_THREADS) k_lz_dots(const double2* __restrict__ basis, long long ld, int nv,
                                                       const double2* __restrict__ w, long long n, double2* __restrict__ partial,
                                                       const LzState* __restrict__ state)
{
    if (state->stop) return;
    const int i0 = blockIdx.y * LZ_GROUP;
    const int cnt = min(LZ_GROUP, nv - i0);
    double re[LZ_GROUP], im[LZ_GROUP];
#pragma unroll
    for (int t = 0; t < LZ_GROUP; ++t) { re[t] = 0.0; im[t] = 0.0; }
    const double2* v0 = basis + (long long)i0 * ld;
    for (long long g = (long long)blockIdx.x * LZ_THREADS + threadIdx.x; g < n; g += (long long)gridDim.x * LZ_THREADS) {
        const double2 b = w[g];
#pragma unroll
        for (int t = 0; t < LZ_GROUP; ++t) {
            if (t < cnt) {
                const double2 a = __ldcs(v0 + (long long)t * ld + g);
                re[t] += a.x * b.x + a.y * b.y;
                im[t] += a.x * b.y - a.y * b.x;
            }
        }
    }
    // block reduction, fixed order: lanes by xor shuffles, then the 8 warps through shared memory
    __shared__ double sre[LZ_THREADS / 32][LZ_GROUP], sim[LZ_THREADS / 32][LZ_GROUP];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int t = 0; t < LZ_GROUP; ++t) {
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) {
            re[t] += __shfl_xor_sync(0xffffffffu, re[t], o);
            im[t] += __shfl_xor_sync(0xffffffffu, im[t], o);
        }
        if (lane == 0) { sre[warp][t] = re[t]; sim[warp][t] = im[t]; }
    }
    __syncthreads();
    if (threadIdx.x < cnt) {
        double r = 0.0, s = 0.0;
        for (int wq = 0; wq < LZ_THREADS / 32; ++wq) { r += sre[wq][threadIdx.x]; s += sim[wq][threadIdx.x]; }
        partial[(long long)blockIdx.x * nv + i0 + threadIdx.x] = make_double2(r, s);
    }
}

// what k_lz_finish does with the summed partials
#define LZ_FIN_NORM0 0                // |v0|^2 -> scale = 1/|v0| (stop if not positive)
#define LZ_FIN_COEF 1                 // coef[i] = sum; alpha[j] (+)= Re coef[j]
#define LZ_FIN_BETA 2                 // beta[j] = sqrt(sum of the norm partials); breakdown test; scale = 1/beta[j]; k_done = j + 1

// coef[i] = sum_b partial[b][i] (fixed order), then the bookkeeping of the step (one block)
__global__ void __launch_bounds__(LZ_MAXK) k_lz_finish(const double2* __restrict__ partial, int nblocks, int nv, double2* __restrict__ coef,
                                                      LzState* __restrict__ state, int what, int j, int first_pass, double breakdown)
{
    if (state->stop) return;
    const int i = threadIdx.x;
    double re = 0.0, im = 0.0;
    if (i < nv) {
        for (int b = 0; b < nblocks; ++b) { const double2 p = partial[(long long)b * nv + i]; re += p.x; im += p.y; }
        if (what == LZ_FIN_COEF) coef[i] = make_double2(re, im);
    }
    if (what == LZ_FIN_COEF && i == j) {
        // the second Gram-Schmidt pass adds the rounding-level correction
        const double a = first_pass ? re : state->alpha[j] + re;
        state->alpha[j] = a;
        if (j == 0) state->alpha0_abs = fabs(a);
    }
    if (what == LZ_FIN_NORM0 && i == 0) {
        if (!(re > 0.0)) state->stop = 2;
        else state->scale = 1.0 / sqrt(re);
    }
    if (what == LZ_FIN_BETA && i == 0) {
        const double b = sqrt(re > 0.0 ? re : 0.0);
        state->beta[j] = b;
        state->k_done = j + 1;
        const double ref = state->alpha0_abs > 1.0 ? state->alpha0_abs : 1.0;
        if (b <= breakdown * ref) state->stop = 1;                      // invariant subspace
        else state->scale = 1.0 / b;
    }
}

// w -= sum_i coef[i] V_i;  npart[blockIdx.x] = sum over the block's elements of |w_new|^2 (as (sum, 0))
__global__ void __launch_bounds__(LZ_THREADS) k_lz_project(const double2* __restrict__ basis, long long ld, int nv,
                                                          const double2* __restrict__ coef, double2* __restrict__ w, long long n,
                                                          double2* __restrict__ npart, const LzState* __restrict__ state)
{
    if (state->stop) return;
    extern __shared__ double2 s_coef[];                                  // [nv]
    for (int i = threadIdx.x; i < nv; i += LZ_THREADS) s_coef[i] = coef[i];
    __syncthreads();
    double nrm = 0.0;
    for (long long g = (long long)blockIdx.x * LZ_THREADS + threadIdx.x; g < n; g += (long long)gridDim.x * LZ_THREADS) {
        double2 x = w[g];
        int i = 0;
        for (; i + 4 <= nv; i += 4) {                                    // four loads in flight
            const double2 v0 = __ldcs(basis + (long long)i * ld + g), v1 = __ldcs(basis + (long long)(i + 1) * ld + g);
            const double2 v2 = __ldcs(basis + (long long)(i + 2) * ld + g), v3 = __ldcs(basis + (long long)(i + 3) * ld + g);
            const double2 c0 = s_coef[i], c1 = s_coef[i + 1], c2 = s_coef[i + 2], c3 = s_coef[i + 3];
            x.x -= c0.x * v0.x - c0.y * v0.y; x.y -= c0.x * v0.y + c0.y * v0.x;
            x.x -= c1.x * v1.x - c1.y * v1.y; x.y -= c1.x * v1.y + c1.y * v1.x;
            x.x -= c2.x * v2.x - c2.y * v2.y; x.y -= c2.x * v2.y + c2.y * v2.x;
            x.x -= c3.x * v3.x - c3.y * v3.y; x.y -= c3.x * v3.y + c3.y * v3.x;
        }
        for (; i < nv; ++i) {
            const double2 c = s_coef[i], v = __ldcs(basis + (long long)i * ld + g);
            x.x -= c.x * v.x - c.y * v.y;
            x.y -= c.x * v.y + c.y * v.x;
        }
        w[g] = x;
        nrm += x.x * x.x + x.y * x.y;
    }
    __shared__ double sn[LZ_THREADS / 32];
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) nrm += __shfl_xor_sync(0xffffffffu, nrm, o);
    if ((threadIdx.x & 31) == 0) sn[threadIdx.x >> 5] = nrm;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int wq = 0; wq < LZ_THREADS / 32; ++wq) s += sn[wq];
        npart[blockIdx.x] = make_double2(s, 0.0);
    }
}

// out = state->scale * in
__global__ void __launch_bounds__(LZ_THREADS) k_lz_scale(const double2* __restrict__ in, double2* __restrict__ out, long long n,
                                                        const LzState* __restrict__ state)
{
    if (state->stop) return;
    const double s = state->scale;
    for (long long g = (long long)blockIdx.x * LZ_THREADS + threadIdx.x; g < n; g += (long long)gridDim.x * LZ_THREADS) {
        const double2 x = in[g];
        out[g] = make_double2(s * x.x, s * x.y);
    }
}

static long long lz_ld(const mcb_space* sp) { return mcb_round_up(sp->nc, 16); }
static long long lz_scratch_bytes(int kmax)
{
    return mcb_round_up(((long long)LZ_BLOCKS + 1) * (kmax + 1) * (long long)sizeof(double2) + LZ_BLOCKS * (long long)sizeof(double2), 256)
           + mcb_round_up((long long)sizeof(LzState), 256);
}

// The paper caps the iteration count at nc / 8; kmax = 0 asks for that cap (at most LZ_MAXK).
static int lz_kmax(const mcb_space* sp, int kmax)
{
    if (kmax != 0) return kmax;
    long long k = sp->nc / 8;
    if (k < 1) k = 1;
    if (k > LZ_MAXK) k = LZ_MAXK;
    if (k > sp->nc) k = sp->nc;
    return (int)k;
}

extern "C" int mcb_lanczos_steps(const mcb_space* sp, int kmax)
{
    if (!sp || kmax < 0 || kmax > LZ_MAXK) return MCB_EINVAL;
    return lz_kmax(sp, kmax);
}

extern "C" long long mcb_lanczos_workspace_bytes(const mcb_space* sp, int kmax)
{
    if (!sp || kmax < 0 || kmax > LZ_MAXK) return MCB_EINVAL;
    kmax = lz_kmax(sp, kmax);
    // (kmax + 1) basis vectors + the work vector w + reduction scratch + state
    return (long long)(kmax + 2) * lz_ld(sp) * (long long)sizeof(double2) + lz_scratch_bytes(kmax);
}

extern "C" int mcb_lanczos(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_v0, int kmax, int mode,
                           double breakdown, double* alpha, double* beta, int* k_done,
                           void* d_workspace, void* d_apply_workspace, void* stream)
{
    if (!sp || !T || !V || !d_v0 || !alpha || !beta || !k_done || !d_workspace) return MCB_EINVAL;
    if (kmax < 0 || kmax > LZ_MAXK) return MCB_EINVAL;
    // kmax = 0 asks for the paper's nc / 8 steps: say so when the library's own cap cut that short
    const bool truncated = kmax == 0 && sp->nc / 8 > LZ_MAXK;
    kmax = lz_kmax(sp, kmax);
    if (((uintptr_t)d_workspace) & 255) return MCB_EINVAL;
    // T, V and the mode are the same for every step: resolve MCB_AUTO once (it inspects the non-zero pattern of T and V) and
    // let the first apply stage the packed coefficients for all the others (coef_hold, mcb_internal.cuh)
    mode = mcb_resolve_mode(sp, T, V, mode);
    if (mode < 0) return mode;
    // a step costs milliseconds on a large space: look at the breakdown flag after every step there, so that no apply is
    // enqueued on a basis slot that was never written; small spaces keep the host out of the way for LZ_SYNC_EVERY steps
    const int sync_every = sp->nc >= (1LL << 20) ? 1 : LZ_SYNC_EVERY;
    cudaStream_t st = (cudaStream_t)stream;
    const long long n = sp->nc, ld = lz_ld(sp);
    double2* basis = (double2*)d_workspace;                              // [kmax + 1][ld]
    double2* w = basis + (long long)(kmax + 1) * ld;
    double2* partial = w + ld;                                           // [LZ_BLOCKS][kmax + 1]
    double2* coef = partial + (long long)LZ_BLOCKS * (kmax + 1);         // [kmax + 1]
    double2* npart = coef + (kmax + 1);                                  // [LZ_BLOCKS]
    LzState* state = (LzState*)((char*)d_workspace + (long long)(kmax + 2) * ld * (long long)sizeof(double2) + lz_scratch_bytes(kmax)
                                - mcb_round_up((long long)sizeof(LzState), 256));
    LzState* h = (LzState*)malloc(sizeof(LzState));
    if (!h) return MCB_ENOMEM;
    int blocks = (int)((n + LZ_THREADS - 1) / LZ_THREADS);
    if (blocks > LZ_BLOCKS) blocks = LZ_BLOCKS;
    *k_done = 0;
    int rc = MCB_OK;
    int launches = 0;
#define LZ_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { rc = mcb_set_cuda_error(e__); goto done; } } while (0)
    LZ_CUDA(cudaMemsetAsync(state, 0, sizeof(LzState), st));
    // v_0 = v0 / |v0|
    k_lz_dots<<<dim3(blocks, 1), LZ_THREADS, 0, st>>>((const double2*)d_v0, ld, 1, (const double2*)d_v0, n, partial, state);
    k_lz_finish<<<1, LZ_MAXK, 0, st>>>(partial, blocks, 1, coef, state, LZ_FIN_NORM0, 0, 1, breakdown);
    k_lz_scale<<<blocks, LZ_THREADS, 0, st>>>((const double2*)d_v0, basis, n, state);
    LZ_CUDA(cudaGetLastError());
    launches += 3;
    sp->coef_hold = 1;
    for (int j = 0; j < kmax; ++j) {
        const int nv = j + 1;
        // (after a breakdown the remaining applies of this batch of LZ_SYNC_EVERY steps still run; their results are not used)
        rc = mcb_hc_apply(sp, T, V, (const mcb_c128*)(basis + (long long)j * ld), (mcb_c128*)w, mode, d_apply_workspace, stream);
        if (rc != MCB_OK) goto done;
        launches += sp->last_launches;
        const dim3 dgrid(blocks, (nv + LZ_GROUP - 1) / LZ_GROUP);
        for (int pass = 0; pass < 2; ++pass) {
            k_lz_dots<<<dgrid, LZ_THREADS, 0, st>>>(basis, ld, nv, w, n, partial, state);
            k_lz_finish<<<1, LZ_MAXK, 0, st>>>(partial, blocks, nv, coef, state, LZ_FIN_COEF, j, pass == 0, breakdown);
            k_lz_project<<<blocks, LZ_THREADS, (size_t)nv * sizeof(double2), st>>>(basis, ld, nv, coef, w, n, npart, state);
            launches += 3;
        }
        k_lz_finish<<<1, LZ_MAXK, 0, st>>>(npart, blocks, 1, coef, state, LZ_FIN_BETA, j, 0, breakdown);
        launches += 1;
        if (j + 1 < kmax) {
            k_lz_scale<<<blocks, LZ_THREADS, 0, st>>>(w, basis + (long long)(j + 1) * ld, n, state);
            launches += 1;
        }
        LZ_CUDA(cudaGetLastError());
        if ((j + 1) % sync_every == 0 && j + 1 < kmax) {              // look at the state: stop issuing work after a breakdown
            LZ_CUDA(cudaMemcpyAsync(&h->scale, &state->scale, sizeof(LzState) - offsetof(LzState, scale), cudaMemcpyDeviceToHost, st));
            LZ_CUDA(cudaStreamSynchronize(st));
            if (h->stop) break;
        }
    }
    LZ_CUDA(cudaMemcpyAsync(h, state, sizeof(LzState), cudaMemcpyDeviceToHost, st));
    LZ_CUDA(cudaStreamSynchronize(st));
    if (h->stop == 2) { rc = MCB_EINVAL; goto done; }                    // v0 has no norm
    *k_done = h->k_done;
    memcpy(alpha, h->alpha, sizeof(double) * (size_t)h->k_done);
    memcpy(beta, h->beta, sizeof(double) * (size_t)h->k_done);
    sp->last_launches = launches;
    if (truncated) rc = MCB_TRUNCATED;
done:
#undef LZ_CUDA
    sp->coef_hold = 0;
    free(h);
    return rc;
}

// ---- host: eigenvalues of the real symmetric tridiagonal matrix tridiag(alpha[0..n-1]; beta[0..n-2]) -----------------
// Sturm-sequence bisection: count(x) = number of eigenvalues below x = number of negative pivots of the LDL^T
// factorisation of T - x I, q_0 = a_0 - x, q_i = a_i - x - b_{i-1}^2 / q_{i-1}; the k-th eigenvalue is bracketed inside the
// Gershgorin interval and bisected down to the last bit.  O(n^2) per spectrum, n <= a few thousand: microseconds to milliseconds.
static int sturm_count(int n, const double* a, const double* b2, double x, double pivmin)
{
    int cnt = 0;
    double q = a[0] - x;
    if (fabs(q) < pivmin) q = -pivmin;
    if (q < 0.0) ++cnt;
    for (int i = 1; i < n; ++i) {
        q = a[i] - x - b2[i - 1] / q;
        if (fabs(q) < pivmin) q = -pivmin;
        if (q < 0.0) ++cnt;
    }
    return cnt;
}

extern "C" int mcb_tridiag_eigvals(int n, const double* alpha, const double* beta, double* eig_out)
{
    if (n < 1 || !alpha || !eig_out || (n > 1 && !beta)) return MCB_EINVAL;
    double* b2 = (double*)malloc(sizeof(double) * (size_t)(n > 1 ? n - 1 : 1));
    if (!b2) return MCB_ENOMEM;
    double lo = alpha[0], hi = alpha[0], bmax = 0.0;
    for (int i = 0; i < n; ++i) {
        const double l = i > 0 ? fabs(beta[i - 1]) : 0.0, r = i + 1 < n ? fabs(beta[i]) : 0.0;
        if (alpha[i] - l - r < lo) lo = alpha[i] - l - r;
        if (alpha[i] + l + r > hi) hi = alpha[i] + l + r;
        if (i + 1 < n) { b2[i] = beta[i] * beta[i]; if (b2[i] > bmax) bmax = b2[i]; }
    }
    const double scale = fabs(lo) > fabs(hi) ? fabs(lo) : fabs(hi);
    const double pivmin = (bmax > 0.0 ? bmax : 1.0) * 2.2250738585072014e-308 * 4.0 + 1e-300;
    const double span = hi - lo;
    lo -= 2.220446049250313e-16 * (scale + span) + pivmin;
    hi += 2.220446049250313e-16 * (scale + span) + pivmin;
    for (int k = 0; k < n; ++k) {
        double l = lo, h = hi;                                          // invariant: count(l) <= k < count(h)
        for (int it = 0; it < 200; ++it) {
            const double mid = 0.5 * (l + h);
            if (!(mid > l && mid < h)) break;                           // adjacent doubles
            if (sturm_count(n, alpha, b2, mid, pivmin) <= k) l = mid; else h = mid;
        }
        eig_out[k] = 0.5 * (l + h);
    }
    free(b2);
    return MCB_OK;
}
