// mcb_internal.cuh -- shared declarations of libmcb (the CUDA product path; nothing here is used by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "mcb.h"

#define MCB_TIMING_RING 512
#define MCB_MAX_APPLY_KERNELS 3
#define MCB_H2D_CHUNKS 16
#define MCB_MAX_M_TILED 12     // up to here the packed coefficient matrix lives on chip (templated kernels); beyond: mcb_apply_big.cu

// ---- device-side view of the small per-space constants -------------------------------------------------
// G[j][s] = binom(s + j, j + 1), j = 0..M-2, s = 0..N: the number of configurations that precede, in the
// order of Eq. (14), every configuration whose prefix sum S_j = n_0 + .. + n_j equals s
// *because of digit j alone*.  With it Algorithm 1's index collapses (hockey stick) to
//     index(n) = nc - 1 - sum_{j=0}^{M-2} G[j][S_j]
// which is what every kernel uses: O(M) look-ups instead of Algorithm 1's O(N) additions.
struct McbDev {
    int N, M;
    int nc, nc1, nc2;          // N_c(N,M), N_c(N-1,M), N_c(N-2,M)
    int ldg;                   // row stride of G (= N + 1)
    const int* G;              // [(M-1)][ldg]   (M == 1: no rows)
    const double* sq;          // sq[j]  = sqrt(j),          j = 0..N+2
    const double* sq2;         // sq2[j] = sqrt(j (j - 1)),  j = 0..N+2   (sq2[0] = sq2[1] = 0)
    int* dbg;                  // [4] debug words (builds with -DMCB_DEBUG_BOUNDS: first out-of-range index, see MCB_CHK)
};

// Bounds checks of our own (compute-sanitizer is not available on every pool): in a -DMCB_DEBUG_BOUNDS build every gather
// and scatter index of the apply / map kernels is checked against its range; the first violation is recorded (site, index)
// in the space's debug words, the access is redirected to element 0, and mcb_debug_bounds() reports it.  Release builds
// compile the checks away.
#ifdef MCB_DEBUG_BOUNDS
#define MCB_CHK(d, idx, n, site) mcb_chk((d).dbg, (long long)(idx), (long long)(n), (site))
__device__ __forceinline__ long long mcb_chk(int* dbg, long long idx, long long n, int site)
{
    if (idx < 0 || idx >= n) {
        if (atomicCAS(dbg, 0, site) == 0) { dbg[1] = (int)idx; dbg[2] = (int)(idx >> 32); }
        return 0;
    }
    return idx;
}
#else
#define MCB_CHK(d, idx, n, site) (idx)
#endif

struct McbFockView {           // hashing table, SoA uint16: occ[j][b], row stride ld
    const uint16_t* occ;       // N-particle space
    long long ld;
    const uint16_t* occ2;      // (N-2)-particle space (NULL if N < 2)
    long long ld2;
};

// Pipelined host apply of the per-output / GEMM modes (mcb_hc_apply_host): outputs and intermediates are cut into slabs by
// the occupation of the last orbital (the most significant digit of the index order): slab k of the outputs only gathers from
// a PREFIX of C, so its kernels can start when that prefix has arrived and its piece of HC can leave while slab k + 1 computes.
#define MCB_MAX_SLABS 16
struct McbSlabs {
    int n;
    long long g_end[MCB_MAX_SLABS];      // outputs of slab k: [g_end[k-1], g_end[k])
    long long m_end[MCB_MAX_SLABS];      // intermediates of slab k: [m_end[k-1], m_end[k]), multiples of 128 (last: nc2)
    cudaEvent_t ev_in[MCB_MAX_SLABS];    // recorded on the copy-in stream when the prefix of C slab k needs is on the device
    cudaEvent_t ev_out[MCB_MAX_SLABS];   // recorded on the compute stream when HC of slab k is complete
};

struct mcb_space {
    int N, M, P;
    int device;
    long long nc, nc1, nc2;
    long long* h_binom;        // (N+1) x (M+1), N_c(n, m)
    void* d_consts;            // one allocation holding G, sq, sq2
    McbDev dev;
    // attached caller-owned structures
    void* d_fock; long long fock_bytes; McbFockView fock;
    int* d_map1;  long long map1_ld;     // [k][l][b], row stride map1_ld
    int* d_map2;  long long map2_ld;     // [ks][ql][b]
    void* d_map2c;                       // compact double-jump map (mcb_map2c.cu)
    // per-apply staging of packed T, V (device, owned)
    void* d_coef; size_t coef_bytes;
    void* h_coef;              // host scratch for packing
    // pinned ring the packed coefficients are uploaded from (mcb_coef_upload): a pageable source would make every apply
    // synchronise with the stream; slot i is reused once the copy recorded in ev_pin[i] has completed
    void* h_pin[4]; cudaEvent_t ev_pin[4]; unsigned pin_next; int pin_state;   // pin_state: 0 not tried, 1 ready, -1 unavailable
    // coefficient hold (mcb_lanczos: T, V and the mode are fixed for a whole run, so only its first apply packs and uploads them)
    //   0: every apply stages its coefficients (default)   1: the next apply stages them and keeps them (-> 2)
    //   2: what is staged (d_coef, runs_coef, the sparse list sizes below) is valid: launchers skip packing and the upload
    int coef_hold;
    int hold_n1, hold_n2; size_t hold_bytes;   // MCB_SPARSE: entry counts and staged bytes of the held list
    int last_launches;
    int n_memcpy, n_memset;    // copies / memsets the last mcb_hc_apply enqueued beside its kernels (mcb_last_apply_memops)
    // per-space launch state (never process-wide: a process may hold spaces on several devices, used by several threads)
    void* runs_coef;           // host scratch of MCB_RUNS: coefficient matrix + packed Vp (lazily allocated)
    int runs_grid;             // persistent grid of k_hc2_runs on this space's device (0: not yet queried)
    int gemm_sms, gemm_ctas_per_sm;      // same for k_hc2_contract
    long long maps2c_grid;     // persistent grid of k_hc_maps2c_group (0: not yet queried; its attribute is set with it)
    size_t sparse_smem_set;    // largest dynamic shared memory size k_hc_sparse has been opted in for on this space's device
    unsigned short* d_pair_ks; // [2][P] pair index -> (k, s), device (M > MCB_MAX_M_TILED only)
    unsigned attr_set;         // bit i: cudaFuncSetAttribute done for kernel family i on this space's device
    // pipelined host apply (mcb_hc_apply_host in MCB_RUNS mode): copy stream, fork/join events, pinned progress values
    cudaStream_t copy_stream;
    cudaEvent_t ev_a, ev_b;
    int* h_prog;               // [MCB_H2D_CHUNKS + 4], pinned; [MCB_H2D_CHUNKS] receives the kernel's error word
    cudaStream_t out_stream;   // copy-out stream of the slab pipeline
    McbSlabs* slabs_store;     // events live here (lazily created)
    const McbSlabs* slabs;     // non-NULL while a pipelined host apply is being enqueued: the launchers cut their work by it
    // optional per-kernel timing (mcb_timing_enable): ring of event tuples, one per apply
    int timing;                          // 0 = off
    int t_count;                         // applies recorded since enable (saturates at MCB_TIMING_RING)
    cudaEvent_t t_ev[MCB_TIMING_RING][MCB_MAX_APPLY_KERNELS + 1];
    int t_launches[MCB_TIMING_RING];
};

static inline long long mcb_round_up(long long x, long long a) { return (x + a - 1) / a * a; }

// error plumbing (mcb_space.cu)
int mcb_set_cuda_error(cudaError_t e);
#define MCB_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return mcb_set_cuda_error(e__); } while (0)
#define MCB_CHECK_LAUNCH() MCB_CUDA(cudaGetLastError())

// ---- pair enumeration (k <= s), order (0,0),(0,1),..,(0,M-1),(1,1),..  (include/mcb.h) ------------------
__host__ __device__ constexpr int mcb_pair_index(int M, int k, int s) { return k * M - k * (k - 1) / 2 + (s - k); }

static inline bool mcb_coef_stale(const mcb_space* sp) { return sp->coef_hold != 2; }
static inline void mcb_coef_staged(mcb_space* sp) { if (sp->coef_hold == 1) sp->coef_hold = 2; }

// packed T, V of this call -> sp->d_coef, asynchronously on st (mcb_space.cu)
int mcb_coef_upload(mcb_space* sp, const void* h_src, size_t bytes, cudaStream_t st);

// implemented per translation unit
int mcb_launch_unrank(const mcb_space* sp, const int* d_idx, long long batch, int* d_occ, cudaStream_t st);
int mcb_launch_rank(const mcb_space* sp, const int* d_occ, long long batch, int* d_idx, cudaStream_t st);
int mcb_launch_fock_table(const mcb_space* sp, int removed, uint16_t* d_out, long long ld, cudaStream_t st);
int mcb_launch_map1(const mcb_space* sp, int* d_out, long long ld, cudaStream_t st);
int mcb_launch_map2(const mcb_space* sp, int* d_out, long long ld, cudaStream_t st);

// ---- hc_apply internals shared by mcb_apply.cu (direct modes) and mcb_apply_gemm.cu (GEMM mode) ----------------
// Vp[a][c] (a = pair(k<=s), c = pair(q<=l)): the bosonic-symmetric part of V, optionally with T folded in
void mcb_pack_pairs(int N, int M, const mcb_c128* T, const mcb_c128* V, bool fold_T, double* vr, double* vi);
long long mcb_gemm_workspace_bytes(const mcb_space* sp);
int mcb_launch_gemm(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_C, mcb_c128* d_HC,
                    void* d_ws, cudaStream_t st);

// MCB_RUNS mode (mcb_apply_runs.cu)
bool mcb_runs_supported(const mcb_space* sp);
long long mcb_runs_workspace_bytes(const mcb_space* sp);
int mcb_launch_runs(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_C, mcb_c128* d_HC,
                   void* d_ws, cudaStream_t st, const mcb_c128* h_C_src = nullptr);

// many orbitals, MCB_MAX_M_TILED < M <= MCB_MAX_M_APPLY (mcb_apply_big.cu)
long long mcb_big_workspace_bytes(const mcb_space* sp);
int mcb_launch_big(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_C, mcb_c128* d_HC, void* d_ws, cudaStream_t st);
long long mcb_big_rho_workspace_bytes(const mcb_space* sp);
int mcb_launch_rho_big(mcb_space* sp, const mcb_c128* d_C, mcb_c128* d_rho1, mcb_c128* d_rho2, void* d_ws, cudaStream_t st);
int mcb_rho_expand_launch(const void* d_G, const mcb_c128* d_C, int N, int M, mcb_c128* d_rho1, mcb_c128* d_rho2, cudaStream_t st);

// compact double-jump map and the MAPS kernel that streams it (mcb_map2c.cu)
long long mcb_map2c_bytes(const mcb_space* sp);
int mcb_launch_map2c(mcb_space* sp, void* d_buf, cudaStream_t st);
int mcb_map2c_export_impl(const mcb_space* sp, long long b0, long long count, long long* host_soff, int* host_entries, long long capacity);
int mcb_launch_maps2c(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_C, mcb_c128* d_HC, cudaStream_t st);
int mcb_pair_tables(mcb_space* sp);

// MCB_SPARSE mode (mcb_apply_sparse.cu)
bool mcb_sparse_preferred(mcb_space* sp, const mcb_c128* T, const mcb_c128* V);
int mcb_launch_sparse(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_C, mcb_c128* d_HC, cudaStream_t st);

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

