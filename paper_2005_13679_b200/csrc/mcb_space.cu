// mcb_space.cu -- space handle, host-side tables, structure attachment, error plumbing.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include "mcb_internal.cuh"

static thread_local int g_last_cuda_error = 0;

int mcb_set_cuda_error(cudaError_t e)
{
    g_last_cuda_error = (int)e;
    (void)cudaGetLastError();            // clear the sticky-free error state
    return MCB_ECUDA;
}

extern "C" int mcb_last_cuda_error(void) { return g_last_cuda_error; }

extern "C" const char* mcb_strerror(int status)
{
    switch (status) {
    case MCB_OK:           return "ok";
    case MCB_TRUNCATED:    return "completed, but with fewer Lanczos steps than the paper's nc / 8 (library cap 1024)";
    case MCB_EINVAL:       return "invalid argument";
    case MCB_ERANGE:       return "configuration space too large for int32 indices (or M > MCB_MAX_M)";
    case MCB_ENOMEM:       return "buffer too small or allocation failed";
    case MCB_ECUDA:        return "CUDA runtime error (see mcb_last_cuda_error)";
    case MCB_ENOTREADY:    return "required structure (hashing table / jump map) not built";
    case MCB_EUNSUPPORTED: return "unsupported for this space (mode unavailable for this M or N)";
    case MCB_ESCRATCH:     return "problem too large for the fixed scratch array of the allocation-free entry point (mcb_rho_static: M > 12)";
    default:               return "unknown status";
    }
}

// Eq. (7) PAPER.md:72 with the convention of Eq. (14) PAPER.md:126.  tab[n][m] = C(n+m-1, m-1) built by
// column recurrence C(n+m-1, m-1) = C(n+m-2, m-1) + C(n+m-2, m-2); entries above 2^62 saturate to 2^62.
static void host_binom(int N, int M, long long* tab)
{
    const long long SAT = 1LL << 62;
    const int W = M + 1;
    for (int n = 0; n <= N; ++n) {
        tab[(size_t)n * W] = 0;
        if (M >= 1) tab[(size_t)n * W + 1] = 1;
    }
    for (int m = 2; m <= M; ++m) {
        tab[m] = 1;                                         // n = 0: the empty configuration
        for (int n = 1; n <= N; ++n) {
            long long up = tab[(size_t)(n - 1) * W + m], left = tab[(size_t)n * W + m - 1];
            tab[(size_t)n * W + m] = (up >= SAT - left) ? SAT : up + left;
        }
    }
}

extern "C" int mcb_space_create(int N, int M, mcb_space** out)
{
    if (!out) return MCB_EINVAL;
    *out = NULL;
    if (N < 1 || M < 1) return MCB_EINVAL;
    if (M > MCB_MAX_M) return MCB_ERANGE;
    mcb_space* sp = new (std::nothrow) mcb_space();
    if (!sp) return MCB_ENOMEM;
    memset(sp, 0, sizeof(*sp));
    sp->N = N; sp->M = M; sp->P = M * (M + 1) / 2;
    sp->h_binom = (long long*)malloc(sizeof(long long) * (size_t)(N + 1) * (M + 1));
    if (!sp->h_binom) { delete sp; return MCB_ENOMEM; }
    host_binom(N, M, sp->h_binom);
    const int W = M + 1;
    sp->nc = sp->h_binom[(size_t)N * W + M];
    sp->nc1 = N >= 1 ? sp->h_binom[(size_t)(N - 1) * W + M] : 0;
    sp->nc2 = N >= 2 ? sp->h_binom[(size_t)(N - 2) * W + M] : 0;
    if (sp->nc >= 2147483647LL) { free(sp->h_binom); delete sp; return MCB_ERANGE; }

    int rc = MCB_OK;
    cudaError_t ce = cudaGetDevice(&sp->device);
    // device constants: G [(M-1)][N+1] int32 | sq [N+3] double | sq2 [N+3] double
    const int ldg = N + 1;
    size_t g_elems = (size_t)(M > 1 ? M - 1 : 0) * ldg;
    size_t g_bytes = (size_t)mcb_round_up((long long)(g_elems * sizeof(int)), 256);
    size_t sq_bytes = (size_t)mcb_round_up((long long)((N + 3) * sizeof(double)), 256);
    size_t total = g_bytes + 2 * sq_bytes + 256;                         // (+ 256: the debug words)
    char* h = (char*)calloc(1, total);
    if (!h) { free(sp->h_binom); delete sp; return MCB_ENOMEM; }
    int* hG = (int*)h;
    // G[j][s] = binom(s+j, j+1) = N_c(s-1, j+2) for s >= 1 (0 for s = 0): the configurations of s-1 particles
    // in j+2 orbitals.  All entries are < nc < 2^31 because s <= N and j + 2 <= M.
    for (int j = 0; j + 2 <= M; ++j)
        for (int s = 0; s <= N; ++s)
            hG[(size_t)j * ldg + s] = s == 0 ? 0 : (int)sp->h_binom[(size_t)(s - 1) * W + (j + 2)];
    double* hsq = (double*)(h + g_bytes);
    double* hsq2 = (double*)(h + g_bytes + sq_bytes);
    for (int j = 0; j <= N + 2; ++j) {
        hsq[j] = sqrt((double)j);
        hsq2[j] = j >= 1 ? sqrt((double)j * (double)(j - 1)) : 0.0;     // j (j-1) < 2^53: exact radicand
    }
    if (ce == cudaSuccess) ce = cudaMalloc(&sp->d_consts, total);
    if (ce == cudaSuccess) ce = cudaMemcpy(sp->d_consts, h, total, cudaMemcpyHostToDevice);
    free(h);
    // packed coefficient staging (largest user: hc_apply GEMM mode): (2P+8) x (2P+4) doubles, x2 for safety
    const size_t P = (size_t)sp->P;
    sp->coef_bytes = (size_t)mcb_round_up((long long)(2 * (2 * P + 8) * (2 * P + 8) * sizeof(double) + 4096), 256);
    if (ce == cudaSuccess) ce = cudaMalloc(&sp->d_coef, sp->coef_bytes);
    sp->h_coef = malloc(sp->coef_bytes);
    if (ce != cudaSuccess) rc = mcb_set_cuda_error(ce);
    else if (!sp->h_coef) rc = MCB_ENOMEM;
    if (rc != MCB_OK) { mcb_space_destroy(sp); return rc; }

    sp->dev.N = N; sp->dev.M = M;
    sp->dev.nc = (int)sp->nc; sp->dev.nc1 = (int)sp->nc1; sp->dev.nc2 = (int)sp->nc2;
    sp->dev.ldg = ldg;
    sp->dev.G = (const int*)sp->d_consts;
    sp->dev.sq = (const double*)((char*)sp->d_consts + g_bytes);
    sp->dev.sq2 = (const double*)((char*)sp->d_consts + g_bytes + sq_bytes);
    sp->dev.dbg = (int*)((char*)sp->d_consts + g_bytes + 2 * sq_bytes);  // zero-initialised with the block
    *out = sp;
    return MCB_OK;
}

extern "C" void mcb_space_destroy(mcb_space* sp)
{
    if (!sp) return;
    for (int i = 0; i < MCB_TIMING_RING; ++i)
        for (int j = 0; j <= MCB_MAX_APPLY_KERNELS; ++j)
            if (sp->t_ev[i][j]) cudaEventDestroy(sp->t_ev[i][j]);
    if (sp->copy_stream) cudaStreamDestroy(sp->copy_stream);
    if (sp->out_stream) cudaStreamDestroy(sp->out_stream);
    if (sp->slabs_store) {
        for (int k = 0; k < MCB_MAX_SLABS; ++k) {
            if (sp->slabs_store->ev_in[k]) cudaEventDestroy(sp->slabs_store->ev_in[k]);
            if (sp->slabs_store->ev_out[k]) cudaEventDestroy(sp->slabs_store->ev_out[k]);
        }
        free(sp->slabs_store);
    }
    if (sp->ev_a) cudaEventDestroy(sp->ev_a);
    if (sp->ev_b) cudaEventDestroy(sp->ev_b);
    if (sp->h_prog) cudaFreeHost(sp->h_prog);
    if (sp->d_consts) cudaFree(sp->d_consts);
    if (sp->d_coef) cudaFree(sp->d_coef);
    if (sp->d_pair_ks) cudaFree(sp->d_pair_ks);
    for (int i = 0; i < 4; ++i) { if (sp->h_pin[i]) cudaFreeHost(sp->h_pin[i]); if (sp->ev_pin[i]) cudaEventDestroy(sp->ev_pin[i]); }
    free(sp->h_coef);
    free(sp->runs_coef);
    free(sp->h_binom);
    delete sp;
}

int mcb_coef_upload(mcb_space* sp, const void* h_src, size_t bytes, cudaStream_t st)
{
    if (bytes > sp->coef_bytes) return MCB_ENOMEM;
    if (sp->pin_state == 0) {
        sp->pin_state = -1;
        if (sp->coef_bytes <= (1u << 20)) {                              // 4 x coef_bytes of pinned memory (4 x 0.45 MB at M = 12)
            bool ok = true;
            for (int i = 0; i < 4 && ok; ++i)
                ok = cudaHostAlloc(&sp->h_pin[i], sp->coef_bytes, cudaHostAllocDefault) == cudaSuccess
                     && cudaEventCreateWithFlags(&sp->ev_pin[i], cudaEventDisableTiming) == cudaSuccess;
            if (ok) sp->pin_state = 1; else (void)cudaGetLastError();
        }
    }
    ++sp->n_memcpy;
    if (sp->pin_state != 1) {                                            // large M: pageable source (the copy synchronises)
        MCB_CUDA(cudaMemcpyAsync(sp->d_coef, h_src, bytes, cudaMemcpyHostToDevice, st));
        return MCB_OK;
    }
    const unsigned slot = sp->pin_next++ & 3u;
    MCB_CUDA(cudaEventSynchronize(sp->ev_pin[slot]));                    // (an event never recorded is complete)
    memcpy(sp->h_pin[slot], h_src, bytes);
    MCB_CUDA(cudaMemcpyAsync(sp->d_coef, sp->h_pin[slot], bytes, cudaMemcpyHostToDevice, st));
    MCB_CUDA(cudaEventRecord(sp->ev_pin[slot], st));
    return MCB_OK;
}

extern "C" long long mcb_nc(const mcb_space* sp) { return sp ? sp->nc : -1; }

extern "C" long long mcb_nc_removed(const mcb_space* sp, int r)
{
    if (!sp || r < 0 || r > 2) return -1;
    return r == 0 ? sp->nc : (r == 1 ? sp->nc1 : sp->nc2);
}

extern "C" int mcb_binom_table(const mcb_space* sp, long long* host_out)
{
    if (!sp || !host_out) return MCB_EINVAL;
    memcpy(host_out, sp->h_binom, sizeof(long long) * (size_t)(sp->N + 1) * (sp->M + 1));
    return MCB_OK;
}

// ---- batched hashing ---------------------------------------------------------------------------------------
extern "C" int mcb_unrank(const mcb_space* sp, const int* d_idx, long long batch, int* d_occ, void* stream)
{
    if (!sp || batch < 0 || (batch > 0 && (!d_idx || !d_occ))) return MCB_EINVAL;
    if (batch == 0) return MCB_OK;
    return mcb_launch_unrank(sp, d_idx, batch, d_occ, (cudaStream_t)stream);
}

extern "C" int mcb_rank(const mcb_space* sp, const int* d_occ, long long batch, int* d_idx, void* stream)
{
    if (!sp || batch < 0 || (batch > 0 && (!d_idx || !d_occ))) return MCB_EINVAL;
    if (batch == 0) return MCB_OK;
    return mcb_launch_rank(sp, d_occ, batch, d_idx, (cudaStream_t)stream);
}

// ---- structures in caller memory ---------------------------------------------------------------------------
static long long fock_ld(long long n) { return mcb_round_up(n > 0 ? n : 1, 128); }

extern "C" long long mcb_structure_bytes(const mcb_space* sp, int which)
{
    if (!sp) return MCB_EINVAL;
    const long long M = sp->M, P = sp->P;
    switch (which) {
    case MCB_FOCK_TABLE:
        return (fock_ld(sp->nc) + (sp->N >= 2 ? fock_ld(sp->nc2) : 0)) * M * (long long)sizeof(uint16_t);
    case MCB_MAP1:
        return mcb_round_up(sp->nc, 64) * M * M * (long long)sizeof(int);
    case MCB_MAP2:
        return mcb_round_up(sp->nc, 64) * P * P * (long long)sizeof(int);
    case MCB_MAP2C:
        if (sp->N < 2) return MCB_EUNSUPPORTED;
        return mcb_map2c_bytes(sp);
    default:
        return MCB_EINVAL;
    }
}

extern "C" int mcb_build_structure(mcb_space* sp, int which, void* d_buf, long long bytes, void* stream)
{
    if (!sp || !d_buf) return MCB_EINVAL;
    long long need = mcb_structure_bytes(sp, which);
    if (need < 0) return (int)need;
    if (bytes < need) return MCB_ENOMEM;
    if (((uintptr_t)d_buf & 255) != 0) return MCB_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    switch (which) {
    case MCB_FOCK_TABLE: {
        if (sp->N > 65535) return MCB_ERANGE;
        uint16_t* p = (uint16_t*)d_buf;
        long long ld = fock_ld(sp->nc), ld2 = fock_ld(sp->nc2);
        rc = mcb_launch_fock_table(sp, 0, p, ld, st);
        if (rc != MCB_OK) return rc;
        uint16_t* p2 = NULL;
        if (sp->N >= 2) {
            p2 = p + ld * sp->M;
            rc = mcb_launch_fock_table(sp, 2, p2, ld2, st);
            if (rc != MCB_OK) return rc;
        }
        sp->d_fock = d_buf; sp->fock_bytes = bytes;
        sp->fock.occ = p; sp->fock.ld = ld; sp->fock.occ2 = p2; sp->fock.ld2 = ld2;
        return MCB_OK;
    }
    case MCB_MAP1: {
        long long ld = mcb_round_up(sp->nc, 64);
        rc = mcb_launch_map1(sp, (int*)d_buf, ld, st);
        if (rc != MCB_OK) return rc;
        sp->d_map1 = (int*)d_buf; sp->map1_ld = ld;
        return MCB_OK;
    }
    case MCB_MAP2: {
        long long ld = mcb_round_up(sp->nc, 64);
        rc = mcb_launch_map2(sp, (int*)d_buf, ld, st);
        if (rc != MCB_OK) return rc;
        sp->d_map2 = (int*)d_buf; sp->map2_ld = ld;
        return MCB_OK;
    }
    case MCB_MAP2C:
        return mcb_launch_map2c(sp, d_buf, st);
    default:
        return MCB_EINVAL;
    }
}

extern "C" int mcb_detach_structure(mcb_space* sp, int which)
{
    if (!sp) return MCB_EINVAL;
    switch (which) {
    case MCB_FOCK_TABLE: sp->d_fock = NULL; sp->fock = McbFockView(); return MCB_OK;
    case MCB_MAP1: sp->d_map1 = NULL; return MCB_OK;
    case MCB_MAP2: sp->d_map2 = NULL; return MCB_OK;
    case MCB_MAP2C: sp->d_map2c = NULL; return MCB_OK;
    default: return MCB_EINVAL;
    }
}

// ---- logical exports (host-side re-layout; test support) -----------------------------------------------------
template <typename TSrc>
static int export_planes(const TSrc* d_base, long long ld, int planes, long long b0, long long count, int* host_out)
{
    // device layout [plane][b] (row stride ld)  ->  host_out[count][planes]
    TSrc* tmp = (TSrc*)malloc(sizeof(TSrc) * (size_t)count);
    if (!tmp) return MCB_ENOMEM;
    cudaError_t e = cudaDeviceSynchronize();
    for (int p = 0; p < planes && e == cudaSuccess; ++p) {
        e = cudaMemcpy(tmp, d_base + (size_t)p * ld + b0, sizeof(TSrc) * (size_t)count, cudaMemcpyDeviceToHost);
        if (e == cudaSuccess)
            for (long long i = 0; i < count; ++i) host_out[(size_t)i * planes + p] = (int)tmp[i];
    }
    free(tmp);
    return e == cudaSuccess ? MCB_OK : mcb_set_cuda_error(e);
}

extern "C" int mcb_fock_export(const mcb_space* sp, int removed, long long b0, long long count, int* host_out)
{
    if (!sp || !host_out || count < 0 || b0 < 0 || (removed != 0 && removed != 2)) return MCB_EINVAL;
    if (!sp->d_fock || (removed == 2 && !sp->fock.occ2)) return MCB_ENOTREADY;
    long long n = removed == 0 ? sp->nc : sp->nc2;
    if (b0 + count > n) return MCB_EINVAL;
    if (count == 0) return MCB_OK;
    return removed == 0 ? export_planes(sp->fock.occ, sp->fock.ld, sp->M, b0, count, host_out)
                        : export_planes(sp->fock.occ2, sp->fock.ld2, sp->M, b0, count, host_out);
}

extern "C" int mcb_map1_export(const mcb_space* sp, long long b0, long long count, int* host_out)
{
    if (!sp || !host_out || count < 0 || b0 < 0 || b0 + count > sp->nc) return MCB_EINVAL;
    if (!sp->d_map1) return MCB_ENOTREADY;
    if (count == 0) return MCB_OK;
    return export_planes(sp->d_map1, sp->map1_ld, sp->M * sp->M, b0, count, host_out);
}

extern "C" int mcb_map2_export(const mcb_space* sp, long long b0, long long count, int* host_out)
{
    if (!sp || !host_out || count < 0 || b0 < 0 || b0 + count > sp->nc) return MCB_EINVAL;
    if (!sp->d_map2) return MCB_ENOTREADY;
    if (count == 0) return MCB_OK;
    return export_planes(sp->d_map2, sp->map2_ld, sp->P * sp->P, b0, count, host_out);
}

extern "C" int mcb_map2c_export(const mcb_space* sp, long long b0, long long count, long long* host_offsets, int* host_entries, long long capacity)
{
    if (!sp || !host_offsets || count < 0 || b0 < 0 || b0 + count > sp->nc || capacity < 0 || (capacity > 0 && !host_entries)) return MCB_EINVAL;
    return mcb_map2c_export_impl(sp, b0, count, host_offsets, host_entries, capacity);
}

extern "C" int mcb_debug_bounds(const mcb_space* sp, long long* host_out)
{
    if (!sp || !host_out) return MCB_EINVAL;
    host_out[0] = 0; host_out[1] = 0;
#ifdef MCB_DEBUG_BOUNDS
    int w[4] = {0, 0, 0, 0};
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(w, sp->dev.dbg, sizeof(w), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return mcb_set_cuda_error(e);
    host_out[0] = w[0];
    host_out[1] = ((long long)w[2] << 32) | (unsigned)w[1];
    return 1;
#else
    return 0;
#endif
}

extern "C" int mcb_last_apply_launches(const mcb_space* sp) { return sp ? sp->last_launches : -1; }

extern "C" int mcb_last_apply_memops(const mcb_space* sp, int* memcpy_out, int* memset_out)
{
    if (!sp || !memcpy_out || !memset_out) return MCB_EINVAL;
    *memcpy_out = sp->n_memcpy; *memset_out = sp->n_memset;
    return MCB_OK;
}

// ---- per-kernel timing of hc_apply (measurement support) ----------------------------------------------------
extern "C" int mcb_timing_enable(mcb_space* sp, int on)
{
    if (!sp) return MCB_EINVAL;
    if (on) {
        for (int i = 0; i < MCB_TIMING_RING; ++i)
            for (int j = 0; j <= MCB_MAX_APPLY_KERNELS; ++j)
                if (!sp->t_ev[i][j]) MCB_CUDA(cudaEventCreate(&sp->t_ev[i][j]));
        sp->t_count = 0;
    }
    sp->timing = on ? 1 : 0;
    return MCB_OK;
}

extern "C" int mcb_timing_read(mcb_space* sp, int max_applies, float* ms_out, int* launches_out)
{
    if (!sp || max_applies < 0 || (max_applies > 0 && (!ms_out || !launches_out))) return MCB_EINVAL;
    int n = sp->t_count < max_applies ? sp->t_count : max_applies;
    for (int i = 0; i < n; ++i) {
        const int L = sp->t_launches[i];
        MCB_CUDA(cudaEventSynchronize(sp->t_ev[i][L]));
        for (int j = 0; j < MCB_MAX_APPLY_KERNELS; ++j) {
            float ms = 0.0f;
            if (j < L) MCB_CUDA(cudaEventElapsedTime(&ms, sp->t_ev[i][j], sp->t_ev[i][j + 1]));
            ms_out[(size_t)i * MCB_MAX_APPLY_KERNELS + j] = ms;
        }
        launches_out[i] = L;
    }
    return n;
}
