// qmcd_dev.cuh -- device-side state, shared-memory carving and small helpers.
// One thread-block CLUSTER of S CTAs LEADS one walker (walkers are
// independent): CTA r of it owns COLUMN slice [N r/S, N (r+1)/S) of every length-N
// vector in the look-ahead (Eq. 3).  The flush (Eq. 4) is cut into row tiles of B that
// are taken, one at a time, by the leader's own CTAs and by the POOL: the CTAs of the
// grid that lead no walker and serve the flush jobs of all of them (qmcd_kernel.cuh).
#pragma once
#include <cuda_runtime.h>
#include <cooperative_groups.h>
#include <stdint.h>

namespace cg = cooperative_groups;

#define QMCD_THREADS 256
#define QMCD_WSTAT_CTAS 512   // CTAs with a slot in QmcdDev::wstat
#define QMCD_WARPS (QMCD_THREADS / 32)

// Status codes mirrored from include/qmcd.h (kept numerically identical).
#define QMCD_DEV_EINVAL (-1)
#define QMCD_DEV_ESINGULAR (-4)

struct QmcdDev {
    int N, K, batch, S;       // S = CTAs per cluster
    int pool;                 // pool CTAs (flush workers serving every walker) in THIS launch, set per launch
    int tile_rows;            // rows of B per flush tile (64 or 128), host choice
    int use_tma;              // host: K <= 64 flush tiles through qmcd_flush_tma.cuh (TMA-fed, 128-row tiles)
    int stagger;              // option: the first window of walker b in a launch is cut short so that the walkers' flushes do not coincide (qmcd_superblock.cuh)
    int la_tma;               // host: qmcd_sweep's blocked look-ahead streams its operands through a TMA ring (qmcd_block.cuh)
    int ldMg;                 // row stride of M in GLOBAL memory: 64 when K <= 64 (a 64 x 64 tile, TMA box), else K
    // ---- flush jobs (leader cluster of walker b -> every worker: its own CTAs and the pool)
    unsigned long long* ticket;   // [batch]  (job number << 32) | next tile; tiles are taken by CAS
    unsigned long long* jdesc;    // [batch]  m | phase << 16 | ntiles << 32 of the posted job
    unsigned* fin;                // [batch]  tiles completed since the launch began
    unsigned* ctrl;               // [4]      [0] = leader clusters that have finished this launch
    double* B;                // [batch][N][N]  inverse, borrowed, updated in place
    double* C;                // [batch][K][N]  queued new columns v_i (one per row)
    double* W;                // [batch][K][N]  rows j_i of the stale inverse B0
    double* Y;                // [batch][K][N]  scratch: Y = M W of Eq. 4 (K > 64, CUDA-core path)
    double* M;                // [batch][ldMg][ldMg]  (I + V'A^-1 U)^-1 = (W C^T)^-1, m x m valid, row stride ldMg
    int* J;                   // [batch][K]     queued electron indices
    int* m;                   // [batch]        queue length
    int* sj;                  // [batch]        staged electron, -1 = none
    double* sR;               // [batch]        staged ratio
    double* sp;               // [batch][K]     staged p (delta term applied)
    double* sc;               // [batch][K]     staged c = M q
    double* sr;               // [batch][K]     staged r = M^T p
    long long* counters;      // [batch][8]     accepted, flushes, cycles: look-ahead, chain, queue append, flush, total; [7] = proposals since the last flush (lock-step)
    long long* fstat;         // [batch][2]     sum of flush ranks, (spare)
    long long* wstat;         // [QMCD_WSTAT_CTAS][4]  per CTA of the grid: flush tiles done, cycles inside tiles, cycles looking for a tile, cycles in the launch
    int* status;              // [4]            sticky: code, walker, move counter
    int flush_path;           // 0 auto, 1 CUDA-core, 2 DMMA
    int mma_smem_ok;          // host: the DMMA flush's shared memory fits
    int m_in_smem;            // host: every CTA keeps its own copy of M in shared memory
    int chain_regs;           // option: blocked look-ahead keeps M in registers when K <= 32
    int blk_ok;               // host: qmcd_sweep may use the blocked look-ahead (qmcd_block.cuh)
    int slot_replace;         // option: an electron accepted again inside one window replaces the column of its queue slot (reading G7, second alternative) instead of flushing first
    int lockstep;             // option: lock-step variant: Eq. 4 every K PROPOSALS; counters[7] = proposals in the window
};

// lock-step option as seen by the kernels (QMCD_NO_LOCKSTEP: A/B build without the variant)
#ifdef QMCD_NO_LOCKSTEP
#define QMCD_LOCKSTEP(P) 0
#else
#define QMCD_LOCKSTEP(P) ((P).lockstep)
#endif

enum QmcdMode { QMCD_MODE_RATIO = 0, QMCD_MODE_ACCEPT = 1, QMCD_MODE_FLUSH = 2, QMCD_MODE_SWEEP = 3 };

struct QmcdArgs {
    QmcdDev P;
    int mode;
    // RATIO
    int j;                        // electron (all walkers) when jv == nullptr
    const int* jv;                // [batch] per-walker electron or nullptr
    const double* v;              // [batch][N]
    double* R_out;                // [batch]
    // ACCEPT
    const unsigned char* mask;    // [batch] or nullptr
    const double* uniforms;       // [batch] or nullptr (Metropolis)
    unsigned char* acc_out;       // [batch] or nullptr
    int accept_all;
    int reject_all;               // qmcd_reject under "lockstep": the proposal still takes a slot
    // SWEEP: v/mask/uniforms/R_out/acc_out are [n_moves][batch]...
    int j_begin, n_moves;
    int blocked;                  // SWEEP: use the blocked look-ahead
};

// Shared-memory carving; every CTA of the cluster has the same layout: a small
// header, then the look-ahead arrays.  The flush (either path) ALIASES everything
// after the header (s.dyn): nothing there is live across a flush (M is written
// back to global memory first, and the queue is empty afterwards).
struct QmcdTmaps;
struct QmcdSmem {
    const QmcdTmaps* tm;   // the kernel's tensor maps (a __grid_constant__ parameter)
    double* red;     // [40]  header: block-reduction scratch (red == start of the CTA's dynamic shared memory)
    int* iflag;      // [16]  header
    unsigned char* dyn;  // start of the aliased region
    double* rs;      // [Ns]  slice of B0[j,:]
    double* vs;      // [Ns]  slice of v
    double* part;    // [2][S][PL] partial p, q, d from every CTA, double buffered by move parity
    double* pf;      // [K]
    double* qf;      // [K]
    double* cf;      // [K]
    double* rf;      // [K]
    double* Ts;      // [QMCD_WARPS][K]  T rows of the CUDA-core flush
    int* Js;         // [K]   queued electron indices (copy of J)
    double* Ms;      // [K][ldM]  this CTA's copy of M (when P.m_in_smem)
};

__host__ __device__ inline int qmcd_slice_lo(int N, int S, int r) { return (int)(((long long)N * r) / S); }
__host__ __device__ inline size_t qmcd_align16(size_t x) { return (x + 15) & ~(size_t)15; }
__host__ __device__ inline int qmcd_PL(int K) { return 2 * K + 2; }
__host__ __device__ inline int qmcd_ldM(int K) { return K | 1; }

#define QMCD_SMEM_HEADER 1024                   // red[40], iflag[16] (384 B); the TMA ring's mbarriers at +512 (qmcd_flush_tma.cuh)

// Bytes after the header: fixed arrays (pf qf cf rf Ts Js [Ms]) followed by a
// union of the per-move look-ahead arrays (rs vs part) and the blocked
// look-ahead's area (blk_bytes, 0 when unused).
__host__ __device__ inline size_t qmcd_smem_fixed_bytes(int K, bool with_M) {
    size_t b = 0;
    b += qmcd_align16((size_t)K * 8) * 4;                      // pf qf cf rf
    b += qmcd_align16((size_t)QMCD_WARPS * K * 8);             // Ts
    b += qmcd_align16((size_t)K * 4);                          // Js
    if (with_M) b += qmcd_align16((size_t)K * qmcd_ldM(K) * 8);  // Ms
    return (b + 127) & ~(size_t)127;                            // the union area starts 128-byte aligned (TMA destination)
}
__host__ __device__ inline size_t qmcd_smem_base_bytes(int N, int K, int S, bool with_M, size_t blk_bytes) {
    size_t ns = (size_t)(N + S - 1) / S + 1;
    size_t u = qmcd_align16(ns * 8) * 2 + qmcd_align16((size_t)2 * S * qmcd_PL(K) * 8);   // rs, vs, part
    if (blk_bytes > u) u = blk_bytes;
    return qmcd_align16(qmcd_smem_fixed_bytes(K, with_M) + u);
}

__device__ inline QmcdSmem qmcd_carve(unsigned char* base, int N, int K, int S, bool with_M) {
    QmcdSmem s;
    size_t ns = (size_t)(N + S - 1) / S + 1;
    unsigned char* p = base;
    s.tm = nullptr;
    s.red = (double*)p; p += 40 * 8;
    s.iflag = (int*)p;
    p = base + QMCD_SMEM_HEADER;
    s.dyn = p;
    s.pf = (double*)p; p += qmcd_align16((size_t)K * 8);
    s.qf = (double*)p; p += qmcd_align16((size_t)K * 8);
    s.cf = (double*)p; p += qmcd_align16((size_t)K * 8);
    s.rf = (double*)p; p += qmcd_align16((size_t)K * 8);
    s.Ts = (double*)p; p += qmcd_align16((size_t)QMCD_WARPS * K * 8);
    s.Js = (int*)p; p += qmcd_align16((size_t)K * 4);
    s.Ms = (double*)p; if (with_M) p += qmcd_align16((size_t)K * qmcd_ldM(K) * 8);
    p = s.dyn + qmcd_smem_fixed_bytes(K, with_M);          // 128-byte aligned
    s.rs = (double*)p; p += qmcd_align16(ns * 8);          // union starts here (blocked area aliases it)
    s.vs = (double*)p; p += qmcd_align16(ns * 8);
    s.part = (double*)p;
    return s;
}

__device__ __forceinline__ double qmcd_warp_sum(double x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// L2-coherent loads for data another CTA of the cluster may have written
// (B rows after a flush, Y, M): bypass the (non-coherent) L1.
__device__ __forceinline__ double qmcd_ldcg(const double* p) { return __ldcg(p); }

__device__ __forceinline__ void qmcd_set_status(const QmcdDev& P, int code, int walker, long long move) {
    if (atomicCAS(P.status, 0, code) == 0) {
        P.status[1] = walker;
        P.status[2] = (int)move;
    }
}

// ---- leader <-> flush workers: words in global memory, release / acquire at gpu scope
__device__ __forceinline__ void qmcd_st_release(unsigned long long* p, unsigned long long v) {
    asm volatile("st.release.gpu.global.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long qmcd_ld_acquire(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned qmcd_ld_acquire32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
