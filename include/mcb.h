/*
 * mcb.h -- C ABI of libmcb: the bosonic Fock-space hot path of Andriati & Gammal, "Hashing algorithms,
 * optimized mappings and massive parallelization of multiconfigurational methods for bosons"
 * (arXiv 2005.13679; citations "PAPER.md:N" are lines of the paper text), hand-written for NVIDIA B200
 * (sm_100a).  One GPU, one process.  No CPU fallback: every entry point that computes runs CUDA kernels.
 *
 * The problem (Eq. 7, 12, 13): N bosons in M orbitals ("IPS") span
 *     nc = N_c(N, M) = binom(N+M-1, M-1)                                     (Eq. 7)
 * configurations |n_0 .. n_{M-1}>, sum n_j = N, enumerated by the combinatorial perfect hash of Sec. III
 * (Eq. 14; Algorithm 1; Algorithm 2), 0-based.
 * Given one- and two-body matrix elements T (M x M) and V (M^4) and a complex vector C of length nc,
 *     HC_g = sum_b <n^g| H |n^b> C_b,
 *     H = sum_{k,l} T[k][l] a+_k a_l + 1/2 sum_{k,s,q,l} V[k][s][q][l] a+_k a+_s a_q a_l     (Eq. 3, 4, 12, 13)
 * is computed without ever storing H.
 *
 * Conventions
 *   - every function returning int returns MCB_OK (0) or a negative MCB_E* code (mcb_lanczos alone may also return the
 *     positive MCB_TRUNCATED, a completed run); nothing throws or aborts.
 *   - "d_" arguments are DEVICE pointers, "h_"/unprefixed array arguments are HOST pointers.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All device work is
 *     enqueued on it and is asynchronous unless stated otherwise.
 *   - the library never allocates or frees caller-visible device memory.  The only device memory it owns
 *     is the constants of the mcb_space (binomial / sqrt tables and the staging of the packed T,V: a few hundred KB up to
 *     12 orbitals, 2 x 16 P^2 bytes beyond -- 18 MB at M = 32), allocated in
 *     mcb_space_create and released in mcb_space_destroy (plus, on the first pipelined mcb_hc_apply_host, two copy
 *     streams, up to 34 events and 80 bytes of pinned host memory; and on the first apply up to 2 MB of pinned host memory
 *     from which the packed T, V are uploaded).  Hashing table, jump maps and apply workspace
 *     live in caller-provided device buffers (e.g. torch tensors) which must stay alive, unmodified,
 *     for as long as the space uses them.
 *   - complex numbers are interleaved (re, im) doubles == C99 double complex == torch.complex128.
 *   - a mcb_space is not thread-safe: calls on one space must be serialised by the caller, and calls on
 *     one space must all use the same stream or be ordered by the caller (T, V are staged per call in a
 *     device buffer owned by the space).
 */
#ifndef MCB_H
#define MCB_H

#ifdef __cplusplus
extern "C" {
#endif

#define MCB_OK            0
#define MCB_EINVAL       -1   /* null pointer, N < 1, M < 1, aliasing, bad enum value                      */
#define MCB_ERANGE       -2   /* nc >= 2^31 - 1 (indices are int32, PAPER.md:268-273 reading A14), M too large */
#define MCB_ENOMEM       -3   /* caller buffer too small / host or device constant allocation failed        */
#define MCB_ECUDA        -4   /* a CUDA runtime call failed; see mcb_last_cuda_error()                       */
#define MCB_ENOTREADY    -5   /* a structure the call needs (hashing table, map) has not been built          */
#define MCB_EUNSUPPORTED -6   /* mode not available for this space (see the hc_apply modes)                    */
#define MCB_TRUNCATED     1   /* the ONE positive status: mcb_lanczos with kmax = 0 completed, but ran fewer steps than the
                                 paper's nc / 8 because of the library's cap of 1024; results are valid       */
#define MCB_ESCRATCH     -7   /* mcb_rho_static: the problem does not fit the library's fixed scratch array (M too large) */

#define MCB_MAX_M        32   /* hashing and map kernels                                                      */
#define MCB_MAX_M_APPLY  32   /* hc_apply, rho, lanczos.  Up to 12 orbitals the packed V (P x P complex, P = M(M+1)/2)
                                 lives on chip and every mode below exists; for 13 <= M <= 32 (the paper's N = 5,
                                 M <= 25 sweep) a generic path serves MCB_AUTO / MCB_GEMM, MCB_SPARSE
                                 has a run-time-M kernel (lattices of more than 12 sites), and the other modes return
                                 MCB_EUNSUPPORTED.  Its workspace is 16 P nc2 bytes (not tiled over the
                                 intermediates): 1.1 GB at N = 10, M = 16, 7.5 GB at N = 10, M = 20, 107 GB at N = 9,
                                 M = 32 -- mcb_apply_workspace_bytes says what a space needs                    */
#define MCB_MAX_M_RUNS    5   /* MCB_RUNS: the embedded coefficient matrix must fit in register fragments      */

/* structures that live in caller-provided device memory (mcb_structure_bytes / mcb_build_structure) */
#define MCB_FOCK_TABLE    0   /* "hashing table" of all occupation vectors, for the N- and
                                 (N-2)-particle spaces; needed by every hc_apply mode                         */
#define MCB_MAP1          1   /* single-jump map                                           */
#define MCB_MAP2          2   /* double-jump map, dense [pair(k<=s)][pair(q<=l)][b] layout  */
#define MCB_MAP2C         3   /* double-jump map in the paper's COMPACT layout (Fig. 3): per
                                 configuration one stride of P targets per ALLOWED removal pair, in the order k = 0..M-1,
                                 s = k..M-1, behind a per-configuration offset: 4 P^2 nc2 bytes + 8 nc.  Needs
                                 FOCK_TABLE built first, N >= 2                                                 */

/* hc_apply modes */
#define MCB_AUTO          0   /* few non-zero elements (at most a quarter of the packed V off its diagonal):
                                 MCB_SPARSE; else N < 2: MCB_REHASH; 2 <= M <= MCB_MAX_M_RUNS and nc >= 2^20:
                                 MCB_RUNS; else MCB_GEMM.  The workspace to provide is that of the dense choice.            */
#define MCB_MAPS          1   /* per-output gather through the stored maps (the paper's fastest CPU/GPU variant,
                                 PAPER.md:238,295).  With the dense planes attached (FOCK_TABLE, MAP1, MAP2): one thread
                                 per configuration.  Without them but with MAP2C (FOCK_TABLE, MAP2C): one thread per
                                 configuration streams its line of the compact table, T riding inside V             */
#define MCB_REHASH        2   /* per-output gather, target indices recomputed on the fly from the hashing table
                                 ("hashing table + algorithm 1" variant); needs FOCK_TABLE       */
#define MCB_GEMM          3   /* on-the-fly rehashing, two-body term factored through the (N-2)-particle space:
                                 W = Vpacked . (F * C[jump]) as an FP64 tensor-core contraction, then a gather;
                                 T folded into V via sum_s a+_s a_s = N.  needs FOCK_TABLE and a workspace     */
#define MCB_RUNS          4   /* the same factorisation for few orbitals (2 <= M <= MCB_MAX_M_RUNS, N >= 2; the
                                 paper's "M = 3..5, N up to 1000" shape): every warp walks a
                                 segment of consecutive (N-2)-particle intermediates (asynchronous gathers, FP64
                                 tensor-core contraction), contributions that stay inside a run of the index
                                 order are pre-summed, then a streaming sum over output-indexed planes.
                                 needs FOCK_TABLE and a workspace                                             */

#define MCB_SPARSE        5   /* structured matrix elements (Lieb-Liniger plane waves, Bose-Hubbard):
                                 per-output gather over the NON-ZERO elements of T and of the packed V only;
                                 diagonal elements (on-site interaction, T_kk) cost no gather.  At most 1024
                                 off-diagonal non-zeros (else MCB_EUNSUPPORTED).  needs FOCK_TABLE, no workspace   */

typedef struct mcb_space mcb_space;          /* opaque */
typedef struct { double re, im; } mcb_c128;

/* ---- space ------------------------------------------------------------------------------------------ */

/* Create the configuration space of N >= 1 bosons in 1 <= M <= MCB_MAX_M orbitals on the CURRENT CUDA
 * device.  Builds the binomial table N_c(n,m) (Eq. 7, 14) on the host and uploads small device constants.
 * MCB_ERANGE if nc >= 2^31 - 1.  *out is set to NULL on failure. */
int  mcb_space_create(int N, int M, mcb_space** out);
void mcb_space_destroy(mcb_space* sp);                        /* NULL is allowed */

long long mcb_nc(const mcb_space* sp);                        /* N_c(N, M); -1 if sp is NULL */
long long mcb_nc_removed(const mcb_space* sp, int r);         /* N_c(N - r, M), r = 0, 1, 2 (0 if N - r < 0) */
/* host_out: (N+1) x (M+1) long long, row-major [n][m]: N_c(n,m) = binom(n+m-1, m-1), N_c(n,0) = 0. */
int  mcb_binom_table(const mcb_space* sp, long long* host_out);

/* ---- batched hashing (Algorithms 1 and 2) ----------------------------------------------------------- */

/* Algorithm 2 for a batch: d_idx int32[batch] -> d_occ int32[batch][M] (row-major).  An index outside
 * [0, nc) yields a row of -1.  batch == 0 is a no-op. */
int  mcb_unrank(const mcb_space* sp, const int* d_idx, long long batch, int* d_occ, void* stream);
/* Algorithm 1 for a batch: d_occ int32[batch][M] -> d_idx int32[batch].  A row with a negative entry or
 * with sum != N yields -1. */
int  mcb_rank(const mcb_space* sp, const int* d_occ, long long batch, int* d_idx, void* stream);

/* ---- hashing table and jump maps (built once per space) ---------------------------- */

/* Bytes the structure needs; < 0 is an MCB_E* code. */
long long mcb_structure_bytes(const mcb_space* sp, int which);
/* Build structure `which` into d_buf (256-byte aligned, at least mcb_structure_bytes) and attach it to the
 * space.  Rebuilding replaces the attachment.  The buffer is owned by the caller. */
int  mcb_build_structure(mcb_space* sp, int which, void* d_buf, long long bytes, void* stream);
/* Detach (the caller is about to free the buffer). */
int  mcb_detach_structure(mcb_space* sp, int which);

/* Logical views for parity tests (synchronous: they synchronise `the build stream` via cudaDeviceSynchronize
 * and copy to host):
 *   fock: host_out int32[count][M]          occupation vector of configurations b0 .. b0+count-1 of the
 *                                           (N - removed)-particle space, removed in {0, 2}
 *   map1: host_out int32[count][M][M]       Map1[b][k][l] = index of n^(b) - e_k + e_l, -1 if n_k = 0;
 *                                           the diagonal k == l is b itself when n_k >= 1
 *   map2: host_out int32[count][P][P]       Map2[b][(k<=s)][(q<=l)] = index of n^(b) - e_k - e_s + e_q + e_l,
 *                                           -1 if the removal is not allowed; pairs ordered (0,0),(0,1),..,
 *                                           (0,M-1),(1,1),..,(M-1,M-1); P = M(M+1)/2 */
int  mcb_fock_export(const mcb_space* sp, int removed, long long b0, long long count, int* host_out);
int  mcb_map1_export(const mcb_space* sp, long long b0, long long count, int* host_out);
int  mcb_map2_export(const mcb_space* sp, long long b0, long long count, int* host_out);
/*   map2c: host_offsets int64[count + 1]   stride offset of lines b0 .. b0 + count (line b holds strides
 *                                           host_offsets[b - b0] .. host_offsets[b - b0 + 1] - 1, one per allowed removal
 *                                           pair (k <= s) in the paper's order)
 *          host_entries int32[..][P]        the strides of those lines, P targets (q <= l) each; `capacity` = int32 elements
 *                                           host_entries can take (MCB_ENOMEM if too small; 0 to fetch the offsets only) */
int  mcb_map2c_export(const mcb_space* sp, long long b0, long long count, long long* host_offsets, int* host_entries, long long capacity);

/* ---- H.C (Eq. 12) ------------------------------------------------------------------------------------- */

/* Device workspace hc_apply needs in `mode` (0 for MCB_MAPS / MCB_REHASH); < 0 is an MCB_E* code. */
long long mcb_apply_workspace_bytes(const mcb_space* sp, int mode);

/* d_HC = H . d_C.
 *   T: host, M*M complex, T[k*M + l] multiplies a+_k a_l (Eq. 3).
 *   V: host, M^4 complex, V[((k*M+s)*M+q)*M+l] multiplies 1/2 a+_k a+_s a_q a_l (Eq. 4, 13).  ANY tensor
 *      is accepted; only its part symmetric under k<->s and q<->l contributes for bosons, and the library
 *      packs exactly that part.  T, V are read before the call returns.
 *   d_C, d_HC: device, nc complex each, 16-byte aligned, must not overlap.
 *   d_workspace: device, mcb_apply_workspace_bytes(sp, mode) bytes, 256-byte aligned (may be NULL if 0).
 * Asynchronous on `stream`.  M must be <= MCB_MAX_M_APPLY (modes other than MCB_AUTO / MCB_GEMM / MCB_SPARSE: M <= 12). */
int  mcb_hc_apply(mcb_space* sp, const mcb_c128* T, const mcb_c128* V,
                  const mcb_c128* d_C, mcb_c128* d_HC, int mode, void* d_workspace, void* stream);

/* The mode mcb_hc_apply(sp, T, V, .., mode, ..) will run: `mode` itself unless it is MCB_AUTO (see MCB_AUTO; depends on
 * the non-zero pattern of T and V) or the space has N < 2 (MCB_GEMM / MCB_RUNS fall back to MCB_REHASH).  < 0 is an
 * MCB_E* code. */
int  mcb_resolve_mode(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, int mode);

/* Same with HOST vectors: copies h_C (nc complex) to d_C_scratch, applies, brings the result to h_HC, and synchronises
 * the stream before returning.  h_C / h_HC should be pinned (and must not overlap).  When the mode resolves to MCB_RUNS and
 * both vectors are pinned the three steps are PIPELINED: C streams in on a stream owned by the space while the kernel,
 * launched at once on `stream`, waits segment by segment for the prefix of C it needs (an intermediate with top occupation
 * j gathers only inside the first nc - N_c(N-j-3, M) elements), and the trailing sum writes HC straight into the mapped
 * host vector.  When it resolves to MCB_GEMM or MCB_SPARSE (M <= 12, nc >= 2^18, both vectors pinned) the work is cut into
 * up to 16 slabs by the occupation of the last orbital: a slab's kernels start when the prefix of C it gathers from has
 * arrived and its piece of HC returns through d_HC_scratch while the next slab computes (two more streams owned by the
 * space).  Otherwise copy, apply, copy run one after the other through d_HC_scratch.  The results are those of mcb_hc_apply,
 * bit for bit.  If, in the MCB_RUNS pipeline, a piece of C does not reach the device within about 4 s (a failed copy) the kernel
 * stops waiting, finishes on what is there, and the call returns MCB_ECUDA with mcb_last_cuda_error() = cudaErrorTimeout (h_HC
 * is then not valid). */
int  mcb_hc_apply_host(mcb_space* sp, const mcb_c128* T, const mcb_c128* V,
                       const mcb_c128* h_C, mcb_c128* h_HC, int mode,
                       mcb_c128* d_C_scratch, mcb_c128* d_HC_scratch, void* d_workspace, void* stream);

/* ---- density matrices (Eq. 10-11; index order of App. B) -------------------------
 *   d_rho1[k*M + l]                 = <Psi| a+_k a_l |Psi>                 (M*M complex, device)
 *   d_rho2[((k*M+s)*M+q)*M + l]     = <Psi| a+_k a+_s a_q a_l |Psi>        (M^4 complex, device; same index order as V,
 *                                                                            so <H> = sum T.rho1 + 1/2 sum V.rho2)
 * for |Psi> = sum_b d_C[b] |n^b> (not normalised by the library).  The two-body matrix is the P x P Gram matrix of
 * the vectors a_q a_l |Psi> over the (N-2)-particle space, accumulated on the FP64 tensor path without atomics
 * (deterministic); rho1 follows from sum_s a+_k a+_s a_s a_l = (N-1) a+_k a_l.  Needs FOCK_TABLE if N >= 2 and
 * mcb_rho_workspace_bytes(sp) bytes of 256-byte aligned device workspace.  M <= MCB_MAX_M_APPLY.  Asynchronous on
 * `stream`; all pointers 16-byte aligned. */
long long mcb_rho_workspace_bytes(const mcb_space* sp);
int  mcb_rho(mcb_space* sp, const mcb_c128* d_C, mcb_c128* d_rho1, mcb_c128* d_rho2, void* d_workspace, void* stream);

/* The same density matrices (Eq. 10-11) for callers that CANNOT ALLOCATE device memory, hence cannot give
 * mcb_rho its workspace: a plug-in that receives C and the result buffers from a host program and has no allocator of its
 * own; a job whose pool claimed the whole device at start-up, so that any further cudaMalloc fails or breaks its memory
 * budget; a time-stepping loop where cudaMalloc / cudaFree are banned because they synchronise the device and block the
 * other streams and threads of the process.  The caller passes the input and the two outputs only; the scratch of the
 * kernels (per-block partial Gram matrices and the reduced P x P matrix) sits in a fixed array of MCB_RHO_STATIC_BYTES
 * inside the library image.  That array costs its size on EVERY GPU that loads libmcb.so, from the first use of the
 * density kernels until the process exits, whether or not this call is ever made.
 *   Limit: M <= MCB_RHO_STATIC_MAX_M (any N the space allows); a larger M returns MCB_ESCRATCH and touches nothing.  When
 *     the array holds fewer partials than mcb_rho's grid has blocks (M = 3..5 and M >= 8) fewer blocks share the work: same
 *     result up to summation order (within the tolerance stated for mcb_rho, bit-identical where the grids agree), slower.
 *   The call itself runs no cudaMalloc / cudaFree / allocating library routine and needs FOCK_TABLE if N >= 2, like mcb_rho.
 *     (mcb_space_create and the FOCK_TABLE buffer are set-up: do them where allocating is still allowed.)
 *   First call on a device: looks up the device address of the array (cudaGetSymbolAddress, which also makes the CUDA
 *     runtime load the kernels' module) and remembers it for that device.  Make that first call during set-up, before any
 *     stream capture is begun.  The space's device must be the current device (MCB_EINVAL otherwise).
 *   Sharing: all spaces, streams and threads of the process use the ONE array of a device.  It keeps the previous call's
 *     contents; nothing needs clearing because each call overwrites every word it later reads.  Two calls whose kernels may
 *     run at the same time on one GPU (different streams, or different host threads) race on it and give wrong results:
 *     order them on one stream or with events.  mcb_rho with caller workspaces has no such restriction.
 * Asynchronous on `stream`; pointers as for mcb_rho. */
#define MCB_RHO_STATIC_MAX_M   12
#define MCB_RHO_STATIC_BYTES   (8 << 20)
int  mcb_rho_static(mcb_space* sp, const mcb_c128* d_C, mcb_c128* d_rho1, mcb_c128* d_rho2, void* stream);

/* ---- Lanczos tridiagonalisation with full re-orthogonalisation -------------------------------
 * Builds, from the start vector d_v0 (device, nc complex, any non-zero norm), the Krylov basis v_0 .. v_k of H in
 * d_workspace and the real tridiagonal coefficients alpha[0..k-1] (diagonal), beta[0..k-1] (beta[j] = |w_j| couples
 * v_j and v_{j+1}; the last one is the residual norm) on the HOST; the eigenvalues of tridiag(alpha, beta[0..k-2])
 * (mcb_tridiag_eigvals) approximate the extremal eigenvalues of H.  Every step is one mcb_hc_apply in `mode` plus a
 * twice-applied classical Gram-Schmidt against all previous vectors (the paper's full re-orthogonalisation); alpha, beta
 * and the breakdown test stay on the device, the host looks at them every 8 steps and at the end.  Stops early when
 * beta[j] <= breakdown * max(1, |alpha[0]|) (invariant subspace); *k_done receives the number of steps taken.
 * 0 <= kmax <= 1024; kmax = 0 takes the paper's iteration cap nc / 8 (at most 1024, at least 1) --
 * mcb_lanczos_steps(sp, kmax) returns the number of steps a given kmax stands for, i.e. the length alpha and beta must have.
 * When nc / 8 > 1024 (e.g. the paper's N = 5, M = 21: 6,641) a kmax = 0 run is cut to 1024 steps -- full re-orthogonalisation
 * over thousands of vectors is not what the device path is sized for -- and the call returns MCB_TRUNCATED (> 0) instead of
 * MCB_OK: alpha, beta and *k_done are valid, the caller is told that the paper's cap was not reached.
 * T and V are packed and uploaded once per call, by its first H.C.
 * d_workspace: mcb_lanczos_workspace_bytes(sp, kmax) bytes, 256-byte aligned ((kmax + 2) vectors + scratch);
 * d_apply_workspace: as for mcb_hc_apply in `mode`.  SYNCHRONOUS (returns after the last step);
 * H must be Hermitian (T, V with the symmetries of BASELINE.json configs) for alpha to be meaningful.
 * MCB_EINVAL also when d_v0 has zero norm. */
int  mcb_lanczos_steps(const mcb_space* sp, int kmax);
long long mcb_lanczos_workspace_bytes(const mcb_space* sp, int kmax);
int  mcb_lanczos(mcb_space* sp, const mcb_c128* T, const mcb_c128* V, const mcb_c128* d_v0, int kmax, int mode,
                 double breakdown, double* alpha, double* beta, int* k_done,
                 void* d_workspace, void* d_apply_workspace, void* stream);

/* Host only: the n eigenvalues, ascending, of the real symmetric tridiagonal matrix with diagonal alpha[0..n-1] and
 * off-diagonal beta[0..n-2] -- the "tridiagonal system ... solved using LAPACK routines" step of the paper's ground-state
 * program, here by Sturm-sequence bisection to the last bit (no LAPACK).  eig_out: n doubles.
 * beta may be NULL when n = 1.  The lowest one, eig_out[0], is the ground-state energy estimate E0. */
int  mcb_tridiag_eigvals(int n, const double* alpha, const double* beta, double* eig_out);

/* Number of kernels the last mcb_hc_apply / mcb_rho on this space launched (for launch accounting). */
int  mcb_last_apply_launches(const mcb_space* sp);
/* Copies and memsets the last mcb_hc_apply on this space enqueued beside its kernels, counted where they are issued (the
 * upload of the packed T, V; the ticket / flag clear of MCB_RUNS).  Host ints. */
int  mcb_last_apply_memops(const mcb_space* sp, int* memcpy_out, int* memset_out);

/* ---- measurement support: device time of each kernel of hc_apply --------------------------------------------
 * mcb_timing_enable(sp, 1) clears the record and makes every following mcb_hc_apply on this space record CUDA
 * events on its stream around each of its kernels (at most 512 applies are kept; later ones are not recorded);
 * mcb_timing_enable(sp, 0) stops recording.  mcb_timing_read waits for the recorded events and writes, for the
 * first min(recorded, max_applies) applies, ms_out[apply][3] (host float, milliseconds of kernel 0, 1, 2 in
 * launch order; 0 for kernels the mode does not launch) and launches_out[apply] (host int).  Returns the
 * number of applies written (>= 0) or an MCB_E* code. */
int  mcb_timing_enable(mcb_space* sp, int on);
int  mcb_timing_read(mcb_space* sp, int max_applies, float* ms_out, int* launches_out);

/* FP64 throughput the current device sustains, measured with register-only kernels on `stream` (synchronous):
 * kind 0 = DFMA chains (plain FP64 pipe), 1 = DMMA m8n8k4 chains (FP64 tensor path), 2 = both interleaved.
 * *tflops_out (host) receives TFLOP/s.  Allocates and frees 8 bytes of device memory internally. */
int  mcb_fp64_peak(int kind, double* tflops_out, void* stream);

/* Debug builds only (nvcc -DMCB_DEBUG_BOUNDS): every gather / scatter index of the apply, map and density kernels is
 * checked against its range on the device.  Synchronises the device and writes host_out[0] = code of the first
 * violating site since the space was created (0: none), host_out[1] = the offending index.  Returns 1 if the checks are
 * compiled in, 0 if not (release build: host_out = {0, 0}), or an MCB_E* code. */
int  mcb_debug_bounds(const mcb_space* sp, long long* host_out);

/* ---- errors ------------------------------------------------------------------------------------------- */
const char* mcb_strerror(int status);
int         mcb_last_cuda_error(void);       /* cudaError_t of the last failing CUDA call in this thread */

#ifdef __cplusplus
}
#endif
#endif /* MCB_H */
