/*
 * qmcd.h -- C-ABI boundary of the B200 (sm_100a) delayed rank-K Slater-inverse
 * update library (arXiv 1708.00744).  Citations are lines of
 * /root/reference/PAPER.md; notation as in DESIGN.md:
 *
 *   N   electrons = matrix order          K  delay
 *   A   Slater matrix, row = orbital, column = electron
 *   B   = A^-1 ("Ainv"), row-major, row j contiguous
 *   j   moved electron (column of A, row of B)
 *   v   the NEW column j of A;  R = det(A_new)/det(A)
 *   m   moves currently queued for a walker, 0 <= m <= K
 *
 * The operation: propose a single-electron move, get its determinant ratio
 * from the STALE inverse plus the Woodbury correction of the <= K queued
 * accepted moves (Eq. 3), accept or reject it, and
 * after K accepted moves rebuild the inverse in one rank-K step (Eq. 4,
 * PAPER.md:84-89).  K = 1 is classic Sherman-Morrison (Eqs. 1-2).
 * `batch` independent walkers are processed together.
 *
 * Conventions common to every call
 *   - All `*_dev` pointers are DEVICE pointers, fp64 unless stated, owned by the
 *     caller (e.g. torch tensors).  The library never allocates device memory
 *     (one exception, outside the method: qmcd_probe_fp64 allocates and frees an
 *     8-byte scratch; the library image itself holds a 1 MiB static device array,
 *     the scratch of qmcd_invert_static).
 *   - Every call only ENQUEUES work on the handle's CUDA stream and returns; no
 *     call synchronises except qmcd_status, qmcd_destroy and qmcd_sweep_host.
 *   - Return value: QMCD_OK (0) or a negative QMCD_E* code.  Argument and state
 *     checks are host-side.  There is NO CPU fallback: without a CUDA device
 *     qmcd_create returns QMCD_ECUDA.
 *   - State machine per handle: IDLE --ratio--> PROPOSED --accept/reject--> IDLE.
 *     A second ratio in PROPOSED replaces the staged proposal.
 */
#ifndef QMCD_H
#define QMCD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define QMCD_OK         0
#define QMCD_EINVAL    (-1)   /* bad argument (range, NULL, size, alignment)       */
#define QMCD_ESTATE    (-2)   /* call not legal in the handle's current state      */
#define QMCD_ECUDA     (-3)   /* CUDA runtime/driver error (see qmcd_strerror)     */
#define QMCD_ESINGULAR (-4)   /* device status: accept of a move with R==0/non-finite */
#define QMCD_ENOMEM    (-5)   /* host allocation failed                             */
#define QMCD_ELIMIT    (-6)   /* size beyond a fixed limit of the entry point (qmcd_invert_static) */

typedef struct qmcd_ctx* qmcd_handle;   /* opaque */

/* Bytes of device workspace qmcd_create needs for (N, K, batch); 0 on bad
 * arguments (N < 1, K < 1, K > N, batch < 1).  Holds the queue of PAPER.md:84:
 * C (queued new columns), W (queued rows of the stale inverse), Y (scratch of
 * Eq. 4), M = (I + V'A^-1 U)^-1 (K x K), J, m and staging. */
size_t qmcd_workspace_bytes(int N, int K, int batch);

/* Create a handle.  workspace_dev: >= qmcd_workspace_bytes bytes, 256-byte
 * aligned, caller-owned, must outlive the handle; it is zero-filled here
 * (enqueued).  cuda_stream: a cudaStream_t (may be NULL = default stream).
 * Errors: QMCD_EINVAL (ranges, K > N, K > 4095, NULL, too small, misaligned), QMCD_ENOMEM
 * (host allocation of the handle failed), QMCD_ECUDA. */
int qmcd_create(qmcd_handle* out, int N, int K, int batch,
                void* workspace_dev, size_t workspace_bytes, void* cuda_stream);

/* Waits for the stream, releases host resources.  NULL is a no-op. */
int qmcd_destroy(qmcd_handle h);

/* Adopt the explicit inverse.  Ainv_dev: [batch][N][N] row-major
 * fp64, 16-byte aligned, BORROWED until the next set_inverse/destroy and
 * updated IN PLACE by every flush.  Resets every walker's queue (m = 0).
 * Errors: QMCD_EINVAL, QMCD_ESTATE (in PROPOSED). */
int qmcd_set_inverse(qmcd_handle h, double* Ainv_dev);

/* Look-ahead determinant ratio (Eqs. 1 and 3) of
 * moving electron j to the position whose orbital column is v, for every
 * walker: R = d - p^T M q with d = B0[j,:].v, p_i = B0[j,:].C[i,:] - delta(j,j_i),
 * q_a = W[a,:].v (m = 0: R = d).  v_dev: [batch][N], read during this call only
 * (the kernel stages a copy).  R_dev: [batch], valid in stream order; signed.
 * Errors: QMCD_EINVAL (j outside [0,N), NULL), QMCD_ESTATE (no inverse set). */
int qmcd_ratio(qmcd_handle h, int j, const double* v_dev, double* R_dev);

/* Same with a per-walker electron index j_dev: [batch] int32 on the device.
 * An index outside [0,N) sets the sticky device status to QMCD_EINVAL. */
int qmcd_ratio_jv(qmcd_handle h, const int* j_dev, const double* v_dev, double* R_dev);

/* Accept the staged proposal for walkers whose mask byte is non-zero, drop it
 * for the others.  mask_dev: [batch] uint8, or NULL = accept all.  An accepted
 * move is queued: M is bordered, (j, v, B0[j,:]) appended, m++.
 * A walker whose m reaches K is flushed here (Eq. 4).  If j is already queued
 * for that walker the queue is flushed first (reading G7).
 * Accepting R == 0 or non-finite sets the sticky status QMCD_ESINGULAR and the
 * move is dropped.  Errors: QMCD_ESTATE (not PROPOSED). */
int qmcd_accept(qmcd_handle h, const unsigned char* mask_dev);

/* Metropolis accept (BASELINE.json configs[2]): walker b accepts iff
 * uniforms_dev[b] < min(1, R_b^2), decided on the device in fp64.
 * acc_out_dev: [batch] uint8 decisions, may be NULL. */
int qmcd_accept_metropolis(qmcd_handle h, const double* uniforms_dev,
                           unsigned char* acc_out_dev);

/* Drop the staged proposal for every walker (== accept with an all-zero mask).
 * Under option "lockstep" the proposal still counts towards the window of K. */
int qmcd_reject(qmcd_handle h);

/* Apply the queue of every walker with m > 0 (Eq. 4):
 * B <- B0 - (B0 C^T - E_J) M W, any rank 1 <= m <= K; m <- 0.  Legal in IDLE
 * only (QMCD_ESTATE otherwise); a no-op for walkers with m == 0. */
int qmcd_flush(qmcd_handle h);

/* Copy the per-walker queue lengths to m_dev: [batch] int32 (enqueued). */
int qmcd_pending(qmcd_handle h, int* m_dev);

/* Synchronise the stream and return the sticky device status in *host_out:
 * 0, QMCD_ESINGULAR or QMCD_EINVAL.  info_out (may be NULL): int[2] =
 * {first offending walker, its move counter}. */
int qmcd_status(qmcd_handle h, int* host_out, int* info_out);

/* Per-walker counters since set_inverse, copied (enqueued) to
 * counters_dev: [batch][8] int64 = {accepted moves, flushes, then SM clock cycles
 * of the walker's leader CTA inside qmcd_sweep: look-ahead products (F1), per-move
 * chain (F1 small part + F2), queue append, flush (F3), whole sweep, proposals in
 * the current window (option "lockstep", else 0)}. */
int qmcd_counters(qmcd_handle h, long long* counters_dev);

/* Measurement aid (not part of the method).  stats_dev: [512][4] int64, one row per CTA of the
 * last qmcd_sweep / qmcd_flush grids since set_inverse (leader clusters first, then the pool):
 * {flush tiles done, SM cycles inside tiles (leader CTAs: inside their flush jobs), cycles looking
 * for a tile (leader CTAs: waiting for tiles taken by others), cycles in the launch}.
 * flush_rank_sum_dev: [batch] int64, the sum of the ranks m of the walker's flushes (with
 * qmcd_counters[.][1] = their number it gives the mean flush rank).  Either may be NULL.  Enqueued. */
int qmcd_worker_stats(qmcd_handle h, long long* stats_dev, long long* flush_rank_sum_dev);

/* Device-resident run of n_moves proposals with no host round trip (the same
 * ratio -> accept -> flush-when-full sequence, one persistent launch; results
 * equal the call-by-call sequence -- bit for bit with options "lookahead" = 1 and "ratio_kernel" = 0,
 * to rounding (another summation order, and an already-queued electron is
 * flushed before its block instead of at its accept) with the default blocked
 * look-ahead, which needs proposals_dev 16-byte aligned; the blocked sweep also
 * flushes a walker's queue up to min(8, K/4) - 1 moves before it is full when the
 * next block would not fit, and may cut a launch's first window short (option "stagger")
 * -- neutral).  Move t proposes electron
 * (j_begin + t) mod N with new column proposals_dev[t][b][:].  Exactly one of
 * mask_dev ([n_moves][batch] uint8) / uniforms_dev ([n_moves][batch] fp64,
 * Metropolis u < min(1,R^2)) is non-NULL.  Outputs R_out_dev [n_moves][batch]
 * fp64 and acc_out_dev [n_moves][batch] uint8 (either may be NULL).  Ends IDLE
 * with moves possibly still queued (no implicit final flush).
 * Errors: QMCD_EINVAL, QMCD_ESTATE (PROPOSED or no inverse). */
int qmcd_sweep(qmcd_handle h, int j_begin, int n_moves,
               const double* proposals_dev, const unsigned char* mask_dev,
               const double* uniforms_dev, double* R_out_dev,
               unsigned char* acc_out_dev);

/* Same run from HOST buffers (end-to-end path): proposals/mask/uniforms are
 * copied host->device in chunks through staging_dev (caller-owned device
 * scratch, >= qmcd_sweep_host_min_staging bytes; larger = bigger chunks),
 * double-buffered against the compute, and R/acc are copied back.  Host
 * buffers should be pinned for overlap.  SYNCHRONISES before returning. */
int qmcd_sweep_host(qmcd_handle h, int j_begin, int n_moves,
                    const double* proposals_host, const unsigned char* mask_host,
                    const double* uniforms_host, double* R_out_host,
                    unsigned char* acc_out_host,
                    void* staging_dev, size_t staging_bytes);
size_t qmcd_sweep_host_min_staging(int N, int batch);

/* Batched on-device inversion (the "explicit copy of the matrix inverse" the
 * method starts from and may refresh): Ainv_dev[b] <- A_dev[b]^-1 for every walker, by
 * Gauss-Jordan elimination with partial pivoting in one cooperative launch -- blocked (panels of 16
 * pivot columns: the matrix crosses HBM N/16 times) when the whole batch is co-resident, else one
 * pass per pivot; the same pivots and arithmetic either way (option "invert_blocked").  A_dev, Ainv_dev:
 * [batch][N][N] row-major fp64 (A: row = orbital, column = electron; may be the same buffer).
 * scratch_dev: caller-owned, 256-byte aligned, >= qmcd_invert_scratch_bytes(N, batch) bytes
 * (0 = N too large for the kernel's shared memory, N <= 14528).  info_dev: [batch] int32, 0 or
 * k+1 of the first zero / non-finite pivot (that walker's result is then garbage); may be NULL.
 * Does not adopt the result: call qmcd_set_inverse(Ainv_dev) afterwards.  Enqueued on the
 * handle's stream.  Errors: QMCD_EINVAL, QMCD_ESTATE (PROPOSED), QMCD_ECUDA. */
size_t qmcd_invert_scratch_bytes(int N, int batch);
int qmcd_invert(qmcd_handle h, const double* A_dev, double* Ainv_dev,
                void* scratch_dev, size_t scratch_bytes, int* info_dev);

/* qmcd_invert for callers that may not allocate device memory at all (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): the same kernel, with its scratch in a file-scope
 * `static __device__` array of qmcd_invert_static_max_bytes() = 1 MiB that every GPU loading the library holds
 * until exit.  Inputs and outputs are still the caller's.  Shapes whose qmcd_invert_scratch_bytes(N, batch)
 * exceed the array are rejected with QMCD_ELIMIT (qmcd_strerror names the sizes); every BASELINE.json shape
 * fits.  The call allocates nothing (no cudaMalloc / cudaFree / allocating library routine) and, like
 * qmcd_invert, only enqueues work on the handle's stream.  ALL calls on a device share the one array, which
 * keeps the last call's contents (this call clears what it uses first): two calls that overlap on the GPU --
 * different streams or handles without an ordering between them -- RACE; serialise them.  The handle's device
 * must be current.  Other errors as qmcd_invert. */
size_t qmcd_invert_static_max_bytes(void);
int qmcd_invert_static(qmcd_handle h, const double* A_dev, double* Ainv_dev, int* info_dev);

/* Tuning / introspection (IDLE only).  set:
 *   "cluster"       CTAs per LEADER cluster (1, 2, 4, 8, 16; other values: QMCD_EINVAL).  Cluster b of the grid leads
 *                   walker b: look-ahead, accept, posting of its flush jobs.
 *   "pool"          -1 auto (default): qmcd_sweep / qmcd_flush launches fill every SM the leader clusters leave free
 *                   with POOL CTAs that take flush tiles of any walker; 0 = leaders only; n > 0 = at most n pool CTAs.
 *                   The pool needs all leader clusters co-resident (else it is 0).  "clusters_per_walker" is the
 *                   round-1 name: 1 = pool off, > 1 = pool auto.
 *   "cooperative"   1 (default): pooled launches are cooperative launches (the driver guarantees co-residency or the
 *                   launch fails, and the step then runs with the leaders alone); 0 = plain launches (profilers that
 *                   cannot replay cooperative cluster launches; safe on an otherwise idle device: one CTA per SM).
 *   "tma"           1 (default): flush tiles for K <= 64, N >= 128, N % 64 == 0 through the TMA-fed kernel
 *                   (128-row tiles); 0 = the cp.async DMMA kernels.  "tile_rows" (64 / 128) applies to the latter.
 *   "la_tma"        1 (default; 2 means the same): qmcd_sweep looks ahead in SUPER-BLOCKS of up to 64 proposals whose
 *                   operands stream through a TMA ring once (K <= 128, K even beyond 64, N >= 128, N % 64 == 0, column
 *                   slices of whole 16- / 8-column chunks); 0 = blocks of 16 proposals with LDG / cp.async strips (the
 *                   path of every other shape).
 *   "stagger"       1: the first window of walker b in a qmcd_sweep launch that starts with empty queues is cut short to
 *                   K (b mod 8 + 1) / 8 accepted moves (flushing early is neutral), so that walkers with
 *                   identical timing do not post their flush jobs in the same instant, window after window.  Default: on for
 *                   2 ... 8 walkers with N >= 2048 (c4), off otherwise; ignored in lock-step.
 *   "invert_blocked" 1 (default): qmcd_invert / qmcd_invert_static run the blocked Gauss-Jordan kernel when the batch is
 *                   co-resident; 0 = the unblocked kernel (one pass over the matrix per pivot).
 *   "ratio_kernel"  1 (default): qmcd_ratio runs the dedicated bandwidth kernel; 0 = the cluster kernel's look-ahead
 *                   (the arithmetic of the per-move sweep, bit for bit).
 *   "flush_path"    0 auto, 1 CUDA-core, 2 DMMA.
 *   "lookahead"     qmcd_sweep: 0 auto = blocked look-ahead when the shape allows (N % (8 cluster) == 0, K <= 152; for
 *                   K > 64 the K x K inverse then stays in global memory, which needs K even; see "la_tma" for the
 *                   super-block variant), 1 = per move.
 *   "slot_replace"  0 (default): accepting an electron that is already queued flushes first (reading G7); 1: it
 *                   replaces the column of its queue slot (M updated by a column-replacement Sherman-Morrison step),
 *                   nothing is flushed; qmcd_sweep then runs the per-move look-ahead.
 *   "lockstep"      0/1: the lock-step variant of PAPER.md:97-99 -- every proposal, accepted or not, takes one of the K
 *                   slots of the window (a rejected one stands for the unchanged column, a zero column of U in Eq. 4, so
 *                   it adds no arithmetic), and Eq. 4 is applied after every K-th PROPOSAL with rank m = the moves
 *                   accepted in the window, 0 <= m <= K: all walkers flush in the same move.  Holds for qmcd_accept* /
 *                   qmcd_reject and the sweeps; qmcd_flush and qmcd_set_inverse open a new window.
 * get: those plus "threads", "smem_bytes", "m_in_smem", "blocked_ok", "max_active_clusters"; "pool" returns the pool
 * CTAs the next sweep / flush launch gets, "tma" / "la_tma" whether that path is active for this handle.
 * get returns the value (>= 0) or a negative error. */
int qmcd_set_option(qmcd_handle h, const char* key, int value);
int qmcd_get_option(qmcd_handle h, const char* key);

/* Roofline denominators measured on this device (not part of the method):
 * kind 0 = register-resident DFMA loop, 1 = register-resident DMMA.8x8x4 loop.
 * Runs on the given stream, synchronises, writes TFLOP/s to *tflops_out. */
int qmcd_probe_fp64(int kind, int iters, void* cuda_stream, double* tflops_out);

const char* qmcd_strerror(int code);
const char* qmcd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* QMCD_H */
