// mcb_lanczos.cu -- Lanczos tridiagonalisation of H with full re-orthogonalisation, device resident
// ("Lanczos tridiagonal decomposition ... with full re-orthogonalisation", the consumer of H.C in
// the paper's ground-state program).
//
//   v_0 = v0 / |v0|;   for j = 0 .. k-1:   w = H v_j                                   (mcb_hc_apply, any mode)
//                                          c_i = <v_i|w>, i <= j;  alpha_j = Re c_j    (k_lz_dots + k_lz_dots_finish)
//                                          w -= sum_{i<=j} c_i v_i   (twice: classical Gram-Schmidt, re-orthogonalised)
//                                          beta_j = |w|;  stop if beta_j <= breakdown * |alpha_0|;  v_{j+1} = w / beta_j
// Orthogonalising against ALL previous vectors removes alpha_j v_j and beta_{j-1} v_{j-1} of the three-term
// recurrence together with the rounding-induced components along older vectors.  alpha, beta go to the host (the
// tridiagonal eigenproblem is solved there, as in the paper); the basis stays in caller-provided device memory.
// All reductions are two-stage with a fixed order (no atomics): the run is bit-reproducible.
#include <math.h>
#include <stdlib.h>
#include "mcb_internal.cuh"

#define LZ_THREADS 256
#define LZ_BLOCKS 592                 // partial sums per dot product (4 per SM on a B200)
#define LZ_MAXK 1024

// partial[b][i] = sum over the block's elements of conj(V_i[g]) w[g], i = 0 .. nv-1 (V_i = basis + i * ld)
__global__ void __launch_bounds__(LZ_THREADS) k_lz_dots(const double2* __restrict__ basis, long long ld, int nv,
                                                       const double2* __restrict__ w, long long n, double2* __restrict__ partial)
{
    __shared__ double sre[LZ_THREADS], sim[LZ_THREADS];
    for (int i = 0; i < nv; ++i) {
        const double2* v = basis + (long long)i * ld;
        double re = 0.0, im = 0.0;
        for (long long g = (long long)blockIdx.x * LZ_THREADS + threadIdx.x; g < n; g += (long long)gridDim.x * LZ_THREADS) {
            const double2 a = v[g], b = w[g];
            re += a.x * b.x + a.y * b.y;
            im += a.x * b.y - a.y * b.x;
        }
        sre[threadIdx.x] = re; sim[threadIdx.x] = im;
        __syncthreads();
        for (int s = LZ_THREADS / 2; s >= 1; s >>= 1) {
            if (threadIdx.x < s) { sre[threadIdx.x] += sre[threadIdx.x + s]; sim[threadIdx.x] += sim[threadIdx.x + s]; }
            __syncthreads();
        }
        if (threadIdx.x == 0) partial[(long long)blockIdx.x * nv + i] = make_double2(sre[0], sim[0]);
        __syncthreads();
    }
}

// coef[i] = sum_b partial[b][i] (fixed order)
__global__ void k_lz_dots_finish(const double2* __restrict__ partial, int nblocks, int nv, double2* __restrict__ coef)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nv) return;
    double re = 0.0, im = 0.0;
    for (int b = 0; b < nblocks; ++b) { const double2 p = partial[(long long)b * nv + i]; re += p.x; im += p.y; }
    coef[i] = make_double2(re, im);
}

// w -= sum_i coef[i] V_i
__global__ void __launch_bounds__(LZ_THREADS) k_lz_project(const double2* __restrict__ basis, long long ld, int nv,
                                                          const double2* __restrict__ coef, double2* __restrict__ w, long long n)
{
    for (long long g = (long long)blockIdx.x * LZ_THREADS + threadIdx.x; g < n; g += (long long)gridDim.x * LZ_THREADS) {
        double2 x = w[g];
        for (int i = 0; i < nv; ++i) {
            const double2 c = coef[i], v = basis[(long long)i * ld + g];
            x.x -= c.x * v.x - c.y * v.y;
            x.y -= c.x * v.y + c.y * v.x;
        }
        w[g] = x;
    }
}

// out = s * in
__global__ void __launch_bounds__(LZ_THREADS) k_lz_scale(const double2* __restrict__ in, double s, double2* __restrict__ out, long long n)
{
    for (long long g = (long long)blockIdx.x * LZ_THREADS + threadIdx.x; g < n; g += (long long)gridDim.x * LZ_THREADS) {
        const double2 x = in[g];
        out[g] = make_double2(s * x.x, s * x.y);
    }
}

static long long lz_ld(const mcb_space* sp) { return mcb_round_up(sp->nc, 16); }
static long long lz_scratch_bytes(int kmax) { return mcb_round_up(((long long)LZ_BLOCKS + 1) * (kmax + 1) * (long long)sizeof(double2), 256); }

extern "C" long long mcb_lanczos_workspace_bytes(const mcb_space* sp, int kmax)
{
    if (!sp || kmax < 1 || kmax > LZ_MAXK) return MCB_EINVAL;
    // (kmax + 1) basis vectors + the work vector w + reduction scratch
    return (long long)(kmax + 2) * lz_ld(sp) * (long long)sizeof(double2) + lz_scratch_bytes(kmax);
}

extern "C" int mcb_lanczos(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_v0, int kmax, int mode,
                           double breakdown, double* alpha, double* beta, int* k_done,
                           void* d_workspace, void* d_apply_workspace, void* stream)
{
    if (!sp || !T || !V || !d_v0 || !alpha || !beta || !k_done || !d_workspace) return MCB_EINVAL;
    if (kmax < 1 || kmax > LZ_MAXK) return MCB_EINVAL;
    if (((uintptr_t)d_workspace) & 255) return MCB_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const long long n = sp->nc, ld = lz_ld(sp);
    double2* basis = (double2*)d_workspace;                              // [kmax + 1][ld]
    double2* w = basis + (long long)(kmax + 1) * ld;
    double2* partial = w + ld;                                           // [LZ_BLOCKS][kmax + 1]
    double2* coef = partial + (long long)LZ_BLOCKS * (kmax + 1);         // [kmax + 1]
    mcb_c128* h = (mcb_c128*)malloc(sizeof(mcb_c128) * (size_t)(kmax + 1));
    if (!h) return MCB_ENOMEM;
    int blocks = (int)((n + LZ_THREADS - 1) / LZ_THREADS);
    if (blocks > LZ_BLOCKS) blocks = LZ_BLOCKS;
    *k_done = 0;
    int rc = MCB_OK;
#define LZ_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { rc = mcb_set_cuda_error(e__); goto done; } } while (0)
    // v_0 = v0 / |v0|
    k_lz_dots<<<blocks, LZ_THREADS, 0, st>>>((const double2*)d_v0, ld, 1, (const double2*)d_v0, n, partial);
    k_lz_dots_finish<<<1, 32, 0, st>>>(partial, blocks, 1, coef);
    LZ_CUDA(cudaGetLastError());
    LZ_CUDA(cudaMemcpyAsync(h, coef, sizeof(mcb_c128), cudaMemcpyDeviceToHost, st));
    LZ_CUDA(cudaStreamSynchronize(st));
    if (!(h[0].re > 0.0)) { rc = MCB_EINVAL; goto done; }
    k_lz_scale<<<blocks, LZ_THREADS, 0, st>>>((const double2*)d_v0, 1.0 / sqrt(h[0].re), basis, n);
    LZ_CUDA(cudaGetLastError());
    for (int j = 0; j < kmax; ++j) {
        const int nv = j + 1;
        rc = mcb_hc_apply(sp, T, V, (const mcb_c128*)(basis + (long long)j * ld), (mcb_c128*)w, mode, d_apply_workspace, stream);
        if (rc != MCB_OK) goto done;
        double a = 0.0;
        for (int pass = 0; pass < 2; ++pass) {
            k_lz_dots<<<blocks, LZ_THREADS, 0, st>>>(basis, ld, nv, w, n, partial);
            k_lz_dots_finish<<<(nv + 127) / 128, 128, 0, st>>>(partial, blocks, nv, coef);
            k_lz_project<<<blocks, LZ_THREADS, 0, st>>>(basis, ld, nv, coef, w, n);
            LZ_CUDA(cudaGetLastError());
            LZ_CUDA(cudaMemcpyAsync(h, coef + j, sizeof(mcb_c128), cudaMemcpyDeviceToHost, st));
            LZ_CUDA(cudaStreamSynchronize(st));
            a += h[0].re;                                                // second pass adds the rounding-level correction
        }
        alpha[j] = a;
        k_lz_dots<<<blocks, LZ_THREADS, 0, st>>>(w, ld, 1, w, n, partial);
        k_lz_dots_finish<<<1, 32, 0, st>>>(partial, blocks, 1, coef);
        LZ_CUDA(cudaGetLastError());
        LZ_CUDA(cudaMemcpyAsync(h, coef, sizeof(mcb_c128), cudaMemcpyDeviceToHost, st));
        LZ_CUDA(cudaStreamSynchronize(st));
        beta[j] = sqrt(h[0].re > 0.0 ? h[0].re : 0.0);
        *k_done = j + 1;
        if (j + 1 == kmax || beta[j] <= breakdown * (fabs(alpha[0]) > 1.0 ? fabs(alpha[0]) : 1.0)) break;   // invariant subspace
        k_lz_scale<<<blocks, LZ_THREADS, 0, st>>>(w, 1.0 / beta[j], basis + (long long)(j + 1) * ld, n);
        LZ_CUDA(cudaGetLastError());
    }
done:
#undef LZ_CUDA
    free(h);
    return rc;
}
