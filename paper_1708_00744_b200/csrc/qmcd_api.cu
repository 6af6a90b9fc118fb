// qmcd_api.cu -- host side of the C-ABI declared in include/qmcd.h: argument and
// state checks, workspace carving, launch policy.  No CPU fallback anywhere.
#include <cuda.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <string.h>
#include <mutex>
#include <new>

#include "../../include/qmcd.h"
#include "qmcd_kernel.cuh"
#include "qmcd_invert.cuh"
#include "qmcd_invert_blocked.cuh"
#include "qmcd_ratio.cuh"

enum { QMCD_IDLE = 0, QMCD_PROPOSED = 1 };

struct qmcd_ctx {
    int N, K, batch;
    cudaStream_t stream;
    cudaStream_t copy_stream;
    cudaEvent_t ev_h2d[2], ev_done[2];
    QmcdDev P;
    int state;
    bool has_inverse;
    size_t smem_bytes;
    int max_cluster;          // largest cluster size the device can co-schedule
    int lookahead;            // qmcd_sweep: 0 auto (blocked when possible), 1 per move
    int pool_opt;             // option "pool": -1 auto (every SM the leaders leave free), 0 off, > 0 that many CTAs
    int coop;                 // option "cooperative": pooled launches ask the driver for co-residency
    QmcdTmaps tmaps;          // 4-D tensor maps of B, C, W, M for the TMA-fed flush (B re-encoded by set_inverse)
    int tile_opt;             // option "tile_rows" for the TMA-fed flush: 0 auto, 64, 128
    int tma_opt;              // option "tma": 1 = use the TMA-fed flush when the shape allows
    bool tmaps_ok;            // C, W, M, Wk encoded (and B, B16 once an inverse is adopted)
    double* rpart; unsigned* rcnt;   // qmcd_ratio kernel scratch
    int ratio_opt;            // option "ratio_kernel": 1 = qmcd_ratio through the dedicated kernel (qmcd_ratio.cuh)
    int invb_opt;             // option "invert_blocked": 1 = qmcd_invert runs the blocked Gauss-Jordan kernel when the batch is co-resident
    int ratio_sms, ratio_res[2];   // SMs and resident CTAs of the ratio kernel's two variants (0 = not queried yet)
    int la_opt;               // option "la_tma": 1 = TMA-ring look-ahead in qmcd_sweep when the shape allows
    bool la_fit;              // the kernel's shared memory was sized with the look-ahead ring
    size_t ctl_off, ctl_bytes;    // job words inside the workspace (zeroed before every pooled launch)
    unsigned char* ws;
    char last_cuda_error[256];
};

static thread_local char g_last_error[256] = "";

static int cuda_fail(qmcd_ctx* h, cudaError_t e, const char* what) {
    snprintf(g_last_error, sizeof(g_last_error), "%s: %s", what, cudaGetErrorString(e));
    if (h) memcpy(h->last_cuda_error, g_last_error, sizeof(g_last_error));
    return QMCD_ECUDA;
}
#define CK(h, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(h, e_, #call); } while (0)

static size_t al256(size_t x) { return (x + 255) & ~(size_t)255; }
static int qmcd_ldMg_host(int K) { return K <= 64 ? 64 : K; }

struct WsLayout { size_t C, W, Y, M, J, m, sj, sR, sp, sc, sr, counters, fstat, wstat, rpart, rcnt, status, ticket, jdesc, fin, ctrl, ctl_end, total; };

static int ratio_gmax(int N) { int g = (N + 63) / 64; return g > 128 ? 128 : g; }

static WsLayout ws_layout(int N, int K, int batch) {
    WsLayout L; size_t o = 0;
    size_t kn = (size_t)batch * K * N * 8;
    L.C = o; o += al256(kn);
    L.W = o; o += al256(kn);
    L.Y = o; o += al256(kn);                                      // Y = M W of Eq. 4 (K > 64 and the CUDA-core flush)
    L.M = o; o += al256((size_t)batch * qmcd_ldMg_host(K) * qmcd_ldMg_host(K) * 8);
    L.J = o; o += al256((size_t)batch * K * 4);
    L.m = o; o += al256((size_t)batch * 4);
    L.sj = o; o += al256((size_t)batch * 4);
    L.sR = o; o += al256((size_t)batch * 8);
    L.sp = o; o += al256((size_t)batch * K * 8);
    L.sc = o; o += al256((size_t)batch * K * 8);
    L.sr = o; o += al256((size_t)batch * K * 8);
    L.counters = o; o += al256((size_t)batch * 8 * 8);
    L.fstat = o; o += al256((size_t)batch * 2 * 8);
    L.wstat = o; o += al256((size_t)QMCD_WSTAT_CTAS * 4 * 8);
    L.rpart = o; o += al256((size_t)batch * ratio_gmax(N) * (2 * (size_t)K + 2) * 8);   // qmcd_ratio partial sums
    L.rcnt = o; o += al256((size_t)batch * 4);
    L.status = o; o += 256;
    L.ticket = o; o += al256((size_t)batch * 8);                  // job words: one block, zeroed per launch
    L.jdesc = o; o += al256((size_t)batch * 8);
    L.fin = o; o += al256((size_t)batch * 4);
    L.ctrl = o; o += 256;
    L.ctl_end = o;
    L.total = o;
    return L;
}

extern "C" size_t qmcd_workspace_bytes(int N, int K, int batch) {
    if (N < 1 || K < 1 || K > N || K > 4095 || batch < 1) return 0;
    return ws_layout(N, K, batch).total;
}

// ---- TMA tensor maps (driver entry point fetched through the runtime: no link against libcuda)
typedef CUresult (*qmcd_encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                   const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static qmcd_encode_fn get_encode_fn() {
    static qmcd_encode_fn fn = nullptr;
    if (!fn) {
        cudaDriverEntryPointQueryResult q;
        void* p = nullptr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
        fn = (qmcd_encode_fn)p;
    }
    return fn;
}
static bool encode_4d(CUtensorMap* tm, const void* base, const cuuint64_t gd[4], const cuuint64_t gs[3], const cuuint32_t bd[4], bool swizzle) {
    qmcd_encode_fn enc = get_encode_fn();
    if (!enc) return false;
    cuuint32_t es[4] = {1, 1, 1, 1};
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<void*>(base), gd, gs, bd, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
               swizzle ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
// A row-major fp64 array [batch][rows][N] seen as {inner, rows, N / inner, batch}: inner = 8 without swizzle
// (an 8 x 8 block of doubles lands as 512 contiguous bytes) or 16 with SWIZZLE_128B; box {inner, box_rows, groups, 1}.
static bool encode_view(CUtensorMap* tm, double* base, int rows, int N, size_t batch_stride_elems, int batch,
                        int inner, int box_rows, int groups, bool swizzle) {
    const cuuint64_t gd[4] = {(cuuint64_t)inner, (cuuint64_t)rows, (cuuint64_t)(N / inner), (cuuint64_t)batch};
    const cuuint64_t gs[3] = {(cuuint64_t)N * 8, (cuuint64_t)inner * 8, (cuuint64_t)batch_stride_elems * 8};
    const cuuint32_t bd[4] = {(cuuint32_t)inner, (cuuint32_t)box_rows, (cuuint32_t)groups, 1};
    return encode_4d(tm, base, gd, gs, bd, swizzle);
}
// The proposals of one qmcd_sweep launch, [n_moves][batch][N], seen as {8, n_moves, N / 8, batch}: row t of walker b
static bool encode_proposals(CUtensorMap* tm, const double* base, int n_moves, int N, int batch, int box_rows, int groups) {
    const cuuint64_t gd[4] = {8, (cuuint64_t)n_moves, (cuuint64_t)(N / 8), (cuuint64_t)batch};
    const cuuint64_t gs[3] = {(cuuint64_t)batch * N * 8, 64, (cuuint64_t)N * 8};
    const cuuint32_t bd[4] = {8, (cuuint32_t)box_rows, (cuuint32_t)groups, 1};
    return encode_4d(tm, base, gd, gs, bd, false);
}
static bool tma_shape_ok(int N, int K) { return K <= 128 && N % 64 == 0 && N >= 128; }
static bool la_shape_ok(int N, int K) { return K <= QMCD_SB_KMAX && N % 64 == 0 && N >= 128; }
static void encode_queue_tmaps(qmcd_ctx* h) {
    h->tmaps_ok = false;
    if (!tma_shape_ok(h->N, h->K)) return;
    const int N = h->N, K = h->K, rows = 8 * qmcd_tma_NB(K);
    const int nq = qmcd_sb_nq(K);
    h->tmaps_ok = encode_view(&h->tmaps.C, h->P.C, K, N, (size_t)K * N, h->batch, 8, rows, 4, false) &&
                  encode_view(&h->tmaps.W32, h->P.W, K, N, (size_t)K * N, h->batch, 8, 32, nq, false) &&
                  encode_view(&h->tmaps.C32, h->P.C, K, N, (size_t)K * N, h->batch, 8, 32, nq, false);
    if (K <= 64)
        h->tmaps_ok = h->tmaps_ok && encode_view(&h->tmaps.W, h->P.W, K, N, (size_t)K * N, h->batch, 16, rows, 2, true) &&
                      encode_view(&h->tmaps.M, h->P.M, 64, 64, (size_t)64 * 64, h->batch, 16, 64, 4, true);
    else                                       // 64 < K <= 128: the tile multiplies by Y = M W (formed by the job's first phase)
        h->tmaps_ok = h->tmaps_ok && encode_view(&h->tmaps.Y, h->P.Y, K, N, (size_t)K * N, h->batch, 16, rows, 2, true);
}
static void refresh_use_tma(qmcd_ctx* h) {
    h->P.use_tma = (h->tma_opt && h->tmaps_ok && h->P.B != nullptr && h->P.mma_smem_ok && h->P.flush_path != 1 &&
                    h->smem_bytes >= qmcd_flush_tma_smem_bytes()) ? 1 : 0;
    // 128-row tiles when a job then still has >= 8 of them, else 64-row tiles (more workers per job: a short flush is
    // latency, not throughput); K > 64 runs 64-row tiles (the registers hold T for 8 rows x 128 columns per warp)
    if (h->P.use_tma) h->P.tile_rows = (h->K <= 64 && h->N >= 1024 && h->tile_opt != 64) || (h->K <= 64 && h->tile_opt == 128) ? 128 : 64;
    h->P.la_tma = (h->la_opt && h->la_fit && h->tmaps_ok && h->P.B != nullptr && h->P.blk_ok) ? 1 : 0;
}

static int configure_kernel(qmcd_ctx* h, int S) {
    const size_t cap = 227 * 1024;
    const int N = h->N, K = h->K;
    // blocked look-ahead: 16-byte vector access to every slice, <= 40 output tiles
    const bool blk_shape = N >= QMCD_TB && (N % (8 * S) == 0) && (2 * ((K + 7) / 8) + 2 <= 8 * QMCD_BLK_MAXU);
    // M in global memory (staged 16 rows at a time, qmcd_blk_xy_global): K even (16-byte rows), small enough for its register tile
    const bool gm_ok = blk_shape && K % 2 == 0 && K <= 16 * QMCD_BLK_YU;
    // super-blocks through the TMA ring (qmcd_superblock.cuh): K <= 128 tensor maps, column slices of whole chunks
    // (measured against the 16-proposal blocks with LDG / cp.async strips: c1 +11 %, c2 +21 %, c3 +8 %, c4 +13 % at K <= 64)
    const bool la_shape = blk_shape && h->la_opt && la_shape_ok(N, K) && N % S == 0 && (N / S) % (8 * qmcd_sb_nq(K)) == 0;
    auto need = [&](bool with_M, size_t blk) { return (size_t)QMCD_SMEM_HEADER + qmcd_smem_base_bytes(N, K, S, with_M, blk); };
    const size_t sbb = qmcd_sb_smem_bytes(K), blkb = qmcd_blk_smem_bytes(K);
    size_t base;
    h->la_fit = false; h->P.m_in_smem = 1; h->P.blk_ok = blk_shape ? 1 : 0;
    if (la_shape && K <= 64 && need(true, sbb) <= cap) { base = need(true, sbb); h->la_fit = true; }                  // super-blocks, M in shared memory
    else if (la_shape && K > 64 && gm_ok && need(false, sbb) <= cap) { base = need(false, sbb); h->la_fit = true; h->P.m_in_smem = 0; }   // ..., M in global memory
    else if (blk_shape && need(true, blkb) <= cap) base = need(true, blkb);                                         // 16-proposal blocks
    else if (gm_ok && need(false, blkb) <= cap) { base = need(false, blkb); h->P.m_in_smem = 0; }                     // ..., M in global memory
    else {                                                                                                          // per-move look-ahead
        h->P.blk_ok = 0;
        base = need(true, 0);
        if (base > cap) { base = need(false, 0); h->P.m_in_smem = 0; }
    }
    const size_t mma = QMCD_SMEM_HEADER + qmcd_flush_mma_smem_bytes(h->N, h->K);
    if (base > cap) { snprintf(g_last_error, sizeof(g_last_error), "shared memory need %zu > 227 KB", base); return QMCD_EINVAL; }
    h->P.mma_smem_ok = (mma <= cap) ? 1 : 0;
    size_t smem = (h->P.mma_smem_ok && mma > base) ? mma : base;
    if (tma_shape_ok(h->N, h->K) && qmcd_flush_tma_smem_bytes() > smem && qmcd_flush_tma_smem_bytes() <= cap) smem = qmcd_flush_tma_smem_bytes();
    // the attribute is per function, not per handle: always allow the device maximum
    CK(h, cudaFuncSetAttribute(qmcd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    CK(h, cudaFuncSetAttribute(qmcd_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    CK(h, cudaFuncSetAttribute(qmcd_kernel_sweep, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    CK(h, cudaFuncSetAttribute(qmcd_kernel_sweep, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    CK(h, cudaFuncSetAttribute(qmcd_kernel_sweep_ls, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    CK(h, cudaFuncSetAttribute(qmcd_kernel_sweep_ls, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    CK(h, cudaFuncSetAttribute(qmcd_kernel_sweep_gm, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    CK(h, cudaFuncSetAttribute(qmcd_kernel_sweep_gm, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    h->smem_bytes = smem;
    h->P.S = S;
    if (h->K > 64) h->P.tile_rows = 64;          // T for 128 rows does not fit beside the chunk ring
    refresh_use_tma(h);
    return QMCD_OK;
}

// Clusters of the current size the device can hold at once (0 on error).
static int max_active_clusters(qmcd_ctx* h, int S, int nclusters) {
    cudaLaunchConfig_t cfg; memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3((unsigned)(nclusters * S)); cfg.blockDim = dim3(QMCD_THREADS);
    cfg.dynamicSmemBytes = h->smem_bytes;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)S; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, qmcd_kernel, &cfg) != cudaSuccess) { (void)cudaGetLastError(); return 0; }
    return n;
}

// Pool CTAs for a launch that may flush: every cluster the device can hold beyond the `batch`
// leader clusters (0 when the leaders alone do not fit at once: a leader waits for its tiles, so
// pool and leaders must be co-resident; the leaders then flush alone, each taking its own tiles).
static int pool_ctas(qmcd_ctx* h) {
    if (h->pool_opt == 0 || !h->P.mma_smem_ok || h->N % 64 != 0 || h->P.flush_path == 1) return 0;
    const int fit = max_active_clusters(h, h->P.S, h->batch + 1);
    int extra = fit - h->batch;
    if (extra < 1) return 0;
    if (h->pool_opt > 0 && extra * h->P.S > h->pool_opt) extra = h->pool_opt / h->P.S;
    return extra * h->P.S;
}

// with_pool: launches that may flush many rows (qmcd_sweep, qmcd_flush) bring the pool along
static int launch(qmcd_ctx* h, QmcdArgs& a, bool with_pool) {
    int pool = with_pool ? pool_ctas(h) : 0;
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.blockDim = dim3(QMCD_THREADS, 1, 1);
    cfg.dynamicSmemBytes = h->smem_bytes;
    cfg.stream = h->stream;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)h->P.S;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    // leaders wait for tiles taken by pool CTAs: ask the driver to guarantee co-residency of the
    // whole grid (the launch fails instead of dead-locking when the device is shared)
    attr[1].id = cudaLaunchAttributeCooperative;
    attr[1].val.cooperative = 1;
    cfg.attrs = attr;
    auto fire = [&]() -> cudaError_t {
        a.P.pool = pool;
        cfg.gridDim = dim3((unsigned)(h->batch * h->P.S + pool), 1, 1);
        cfg.numAttrs = (pool > 0 && h->coop) ? 2 : 1;
        cudaError_t e = cudaMemsetAsync(h->ws + h->ctl_off, 0, h->ctl_bytes, h->stream);   // job words of this launch
        if (e != cudaSuccess) return e;
        if (a.mode == QMCD_MODE_SWEEP && a.blocked && !h->P.m_in_smem)
            return cudaLaunchKernelEx(&cfg, qmcd_kernel_sweep_gm, a, h->tmaps);
        if (a.mode == QMCD_MODE_SWEEP && a.blocked)
            return h->P.lockstep ? cudaLaunchKernelEx(&cfg, qmcd_kernel_sweep_ls, a, h->tmaps) : cudaLaunchKernelEx(&cfg, qmcd_kernel_sweep, a, h->tmaps);
        return cudaLaunchKernelEx(&cfg, qmcd_kernel, a, h->tmaps);
    };
    cudaError_t e = fire();
    if (e != cudaSuccess && pool > 0) {
        // the pool is an optimisation: when the cooperative launch is refused (device shared with
        // other work) run the same step with the leader clusters alone
        (void)cudaGetLastError();
        pool = 0;
        e = fire();
    }
    if (e != cudaSuccess) return cuda_fail(h, e, "cudaLaunchKernelEx");
    return QMCD_OK;
}

// CTAs per leader cluster.  The look-ahead of a walker is a latency chain on its leader cluster
// (strips: ~N (2m + 32) 8 / S bytes per CTA and block of 16 proposals; then ~1100 cycles per move
// that do not shrink with S), while flush tiles go to any free CTA.  With many walkers the pool
// hides one walker's look-ahead behind the others' flushes, so small clusters (more pool CTAs,
// no DSMEM exchange) win; with few walkers the chain is exposed and a larger S shortens it.
static int default_S(int N, int K, int batch, int cap) {
    // measured with the super-block look-ahead (K = 64, 99 % acceptance, fraction of the DMMA peak for S = 1/2/4/8/16):
    // 1 walker N = 2048: .058/.065/.070/.072/.073, N = 8192: .26/.29/.32/.34/.34; 4 walkers N = 2048: .22/.24/.26/.27;
    // 16 walkers N = 1024: .38/.39/.41, N = 512 (c1, K = 32): .18/.19/.20, N = 2048: .84/.80; 8 walkers N = 4096 (c4) with
    // staggered windows: .87/.86/.72 at 99 % acceptance but .57/.69/.66 at 50 % and .36/.40/.40 at K = 16 -- the look-ahead of a
    // window is long against a tile there, so clusters of 2; 32 and 64 walkers (c3, c2): the pool hides the look-ahead, S = 1
    int s = 1;
    if (K <= 64) {
        if (batch <= 4) s = 8; else if (batch <= 16) s = 4;
        if (batch > 4 && (long long)N * batch >= 32768) s = (batch <= 8) ? 2 : 1;    // (c4: 2, with staggered windows, see qmcd_create; 16 x 2048: 1)
    } else {                                       // the 16-proposal blocks of qmcd_block.cuh / the per-move look-ahead
        if (batch <= 4) s = 8; else if (batch <= 16) s = 2;
        if ((long long)N * batch <= 16384) s *= 2;
    }
    // K > 152 (or odd K > 64) runs the per-move look-ahead (one cluster barrier per proposal, 2m + 2 streamed rows): a
    // latency chain that shortens with S (measured with it: c3 K=128 S=1/2/4 -> 0.27/0.38/0.33 of the DMMA peak; c4 K=256
    // S=2/4/8 -> 0.12/0.16/0.18).  64 < K <= 152, K even, keeps the blocked look-ahead with M in global memory (c3 K=128
    // S=1/2/4 -> 0.48/0.46/0.39; c4 K=128 S=1/2/4 -> 0.41/0.51/0.45) and the cluster size of the small delays.
    if (K > 152 || (K > 64 && (K & 1))) s *= (K > 128) ? 4 : 2;
    while (s > 1 && (N / s < 64 || N % (8 * s) != 0)) s /= 2;
    if (s > cap) s = cap;
    return s < 1 ? 1 : s;
}

extern "C" int qmcd_create(qmcd_handle* out, int N, int K, int batch,
                           void* workspace_dev, size_t workspace_bytes, void* cuda_stream) {
    if (!out) return QMCD_EINVAL;
    *out = nullptr;
    size_t need = qmcd_workspace_bytes(N, K, batch);
    if (need == 0 || !workspace_dev || workspace_bytes < need || ((uintptr_t)workspace_dev & 255)) return QMCD_EINVAL;
    int dev = 0;
    CK(nullptr, cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CK(nullptr, cudaGetDeviceProperties(&prop, dev));
    if (prop.major < 10) { snprintf(g_last_error, sizeof(g_last_error), "device sm_%d%d is not Blackwell (sm_100a build)", prop.major, prop.minor); return QMCD_ECUDA; }
    qmcd_ctx* h = new (std::nothrow) qmcd_ctx();
    if (!h) return QMCD_ENOMEM;
    memset(h, 0, sizeof(*h));
    h->N = N; h->K = K; h->batch = batch;
    h->stream = (cudaStream_t)cuda_stream;
    h->state = QMCD_IDLE;
    unsigned char* ws = (unsigned char*)workspace_dev;
    WsLayout L = ws_layout(N, K, batch);
    h->ws = ws; h->ctl_off = L.ticket; h->ctl_bytes = L.ctl_end - L.ticket;
    h->pool_opt = -1; h->coop = 1;
    QmcdDev& P = h->P;
    P.N = N; P.K = K; P.batch = batch; P.S = 1; P.B = nullptr;
    P.C = (double*)(ws + L.C); P.W = (double*)(ws + L.W); P.Y = (double*)(ws + L.Y);
    P.M = (double*)(ws + L.M); P.J = (int*)(ws + L.J); P.m = (int*)(ws + L.m);
    P.sj = (int*)(ws + L.sj); P.sR = (double*)(ws + L.sR);
    P.sp = (double*)(ws + L.sp); P.sc = (double*)(ws + L.sc); P.sr = (double*)(ws + L.sr);
    P.counters = (long long*)(ws + L.counters); P.fstat = (long long*)(ws + L.fstat); P.wstat = (long long*)(ws + L.wstat); P.status = (int*)(ws + L.status);
    P.ticket = (unsigned long long*)(ws + L.ticket); P.jdesc = (unsigned long long*)(ws + L.jdesc);
    P.fin = (unsigned*)(ws + L.fin); P.ctrl = (unsigned*)(ws + L.ctrl);
    P.chain_regs = 1; P.pool = 0;
    // staggered first windows (qmcd_superblock.cuh): few walkers with long tiles lock their flushes in step otherwise (c4, clusters of
    // 2: 0.64 -> 0.85 of the DMMA peak; clusters of 1: 0.83 -> 0.86); with many walkers or short tiles the extra low-rank flush per
    // walker and launch only costs (c1 -3 %, c2 -2 %, c3 and 16 x 2048: 0)
    P.stagger = (batch >= 2 && batch <= 8 && N >= 2048) ? 1 : 0;
    P.flush_path = 0; P.use_tma = 0; P.ldMg = qmcd_ldMg_host(K);
    h->tma_opt = 1; h->la_opt = 1; h->la_fit = false; h->ratio_opt = 1; h->invb_opt = 1;
    h->rpart = (double*)(ws + L.rpart); h->rcnt = (unsigned*)(ws + L.rcnt);
    encode_queue_tmaps(h);
    P.tile_rows = (K <= 64 && N >= 2048) ? 128 : 64;
    int rc = QMCD_OK;
    do {
        cudaError_t e = cudaMemsetAsync(ws, 0, L.total, h->stream);
        if (e != cudaSuccess) { rc = cuda_fail(h, e, "cudaMemsetAsync(workspace)"); break; }
        e = cudaMemsetAsync(P.sj, 0xff, (size_t)batch * 4, h->stream);
        if (e != cudaSuccess) { rc = cuda_fail(h, e, "cudaMemsetAsync(sj)"); break; }
        e = cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) { rc = cuda_fail(h, e, "cudaStreamCreate"); break; }
        for (int i = 0; i < 2 && rc == QMCD_OK; ++i) {
            if ((e = cudaEventCreateWithFlags(&h->ev_h2d[i], cudaEventDisableTiming)) != cudaSuccess) rc = cuda_fail(h, e, "cudaEventCreate");
            else if ((e = cudaEventCreateWithFlags(&h->ev_done[i], cudaEventDisableTiming)) != cudaSuccess) rc = cuda_fail(h, e, "cudaEventCreate");
        }
        if (rc != QMCD_OK) break;
        h->max_cluster = 16;
        // S = CTAs per leader cluster: the default of default_S, halved until `batch` clusters of it
        // are co-resident (so that a pool can be attached) or S = 1
        int S = default_S(N, K, batch, h->max_cluster);
        for (;; S /= 2) {
            rc = configure_kernel(h, S);
            if (rc != QMCD_OK || S == 1) break;
            if (max_active_clusters(h, S, batch) >= batch) break;
        }
    } while (0);
    if (rc != QMCD_OK) {
        if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
        for (int i = 0; i < 2; ++i) { if (h->ev_h2d[i]) cudaEventDestroy(h->ev_h2d[i]); if (h->ev_done[i]) cudaEventDestroy(h->ev_done[i]); }
        delete h;
        return rc;
    }
    *out = h;
    return QMCD_OK;
}

extern "C" int qmcd_destroy(qmcd_handle h) {
    if (!h) return QMCD_OK;
    cudaStreamSynchronize(h->stream);
    cudaStreamSynchronize(h->copy_stream);
    cudaStreamDestroy(h->copy_stream);
    for (int i = 0; i < 2; ++i) { cudaEventDestroy(h->ev_h2d[i]); cudaEventDestroy(h->ev_done[i]); }
    delete h;
    return QMCD_OK;
}

extern "C" int qmcd_set_inverse(qmcd_handle h, double* Ainv_dev) {
    if (!h || !Ainv_dev || ((uintptr_t)Ainv_dev & 15)) return QMCD_EINVAL;
    if (h->state != QMCD_IDLE) return QMCD_ESTATE;
    h->P.B = Ainv_dev;
    if (h->tmaps_ok && !(encode_view(&h->tmaps.B, Ainv_dev, h->N, h->N, (size_t)h->N * h->N, h->batch, 8, 128, 4, false) &&
                         encode_view(&h->tmaps.B64, Ainv_dev, h->N, h->N, (size_t)h->N * h->N, h->batch, 8, 64, 4, false) &&
                         encode_view(&h->tmaps.Bs[0], Ainv_dev, h->N, h->N, (size_t)h->N * h->N, h->batch, 8, 16, qmcd_sb_nq(h->K), false) &&
                         encode_view(&h->tmaps.Bs[1], Ainv_dev, h->N, h->N, (size_t)h->N * h->N, h->batch, 8, 32, qmcd_sb_nq(h->K), false) &&
                         encode_view(&h->tmaps.Bs[2], Ainv_dev, h->N, h->N, (size_t)h->N * h->N, h->batch, 8, 64, qmcd_sb_nq(h->K), false)))
        h->tmaps_ok = false;
    refresh_use_tma(h);
    CK(h, cudaMemsetAsync(h->P.m, 0, (size_t)h->batch * 4, h->stream));
    CK(h, cudaMemsetAsync(h->P.sj, 0xff, (size_t)h->batch * 4, h->stream));
    CK(h, cudaMemsetAsync(h->P.counters, 0, (size_t)h->batch * 64, h->stream));
    CK(h, cudaMemsetAsync(h->P.fstat, 0, (size_t)h->batch * 16, h->stream));
    CK(h, cudaMemsetAsync(h->P.wstat, 0, (size_t)QMCD_WSTAT_CTAS * 32, h->stream));
    CK(h, cudaMemsetAsync(h->P.status, 0, 16, h->stream));
    h->has_inverse = true;
    return QMCD_OK;
}

static QmcdArgs base_args(qmcd_ctx* h, int mode) {
    QmcdArgs a;
    memset(&a, 0, sizeof(a));
    a.P = h->P;
    a.mode = mode;
    return a;
}

// The dedicated ratio kernel: column slices of 32 NU VEC columns (NU = 4 or 2 vectors per lane and row) x GR groups of queue rows,
// chosen so that the grid is ONE wave of resident CTAs, as full as possible (measured on c3 shapes: 1024 CTAs in 2.3 waves 23 us,
// one wave ~15 us: every wave pays the kernel's chain of dependent memory round trips again).
template <int VEC, int NU>
static int launch_ratio_t(qmcd_ctx* h, QmcdRatioArgs& a, int sms, int* resident_out, bool fire) {
    const size_t smem = (size_t)4 * h->K * 8;
    if (smem > 48 * 1024) CK(h, cudaFuncSetAttribute(qmcd_ratio_kernel<VEC, NU>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (!fire) {
        int per_sm = 0;
        CK(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, qmcd_ratio_kernel<VEC, NU>, QMCD_THREADS, smem));
        *resident_out = per_sm * sms;
        return QMCD_OK;
    }
    dim3 grid((unsigned)a.G, (unsigned)a.GR, (unsigned)h->batch);
    qmcd_ratio_kernel<VEC, NU><<<grid, QMCD_THREADS, smem, h->stream>>>(a);
    CK(h, cudaGetLastError());
    return QMCD_OK;
}
static int launch_ratio(qmcd_ctx* h, int j, const int* jv, const double* v_dev, double* R_dev) {
    const int N = h->N, K = h->K;
    const bool vec2 = (N % 2 == 0) && (((uintptr_t)v_dev & 15) == 0);
    const int per = 32 * (vec2 ? 2 : 1);                 // columns per lane round
    const int gmax = ratio_gmax(N);
    QmcdRatioArgs a;
    a.P = h->P; a.j = j; a.jv = jv; a.v = v_dev; a.R_out = R_dev; a.part = h->rpart; a.cnt = h->rcnt;
    if (h->ratio_sms == 0) {                             // once per handle: resident CTAs of the two variants
        int dev = 0;
        CK(h, cudaGetDevice(&dev));
        CK(h, cudaDeviceGetAttribute(&h->ratio_sms, cudaDevAttrMultiProcessorCount, dev));
        int rc = vec2 ? launch_ratio_t<2, 4>(h, a, h->ratio_sms, &h->ratio_res[0], false) : launch_ratio_t<1, 4>(h, a, h->ratio_sms, &h->ratio_res[0], false);
        if (rc == QMCD_OK) rc = vec2 ? launch_ratio_t<2, 2>(h, a, h->ratio_sms, &h->ratio_res[1], false) : launch_ratio_t<1, 2>(h, a, h->ratio_sms, &h->ratio_res[1], false);
        if (rc != QMCD_OK) { h->ratio_sms = 0; return rc; }
    }
    // candidates (NU, GR): the largest grid that is still one wave; ties -> wider slices (fewer partial sums)
    int bestNU = 0, bestGR = 1, bestG = 0, best_ctas = -1;
    for (int v = 0; v < 2; ++v) {
        const int NU = v ? 2 : 4, slice = NU * per;
        int G = (N + slice - 1) / slice;
        if (G > gmax) continue;
        for (int GR = 1; GR <= 8; GR *= 2) {
            if (GR > 1 && 8 * (GR / 2) >= K) break;     // no more row groups than rows
            const long long ctas = (long long)h->batch * G * GR;
            if (ctas <= h->ratio_res[v] && ctas > best_ctas) { best_ctas = (int)ctas; bestNU = NU; bestGR = GR; bestG = G; }
        }
    }
    if (bestNU == 0) {                                   // even the smallest grid is more than a wave (many walkers): widest slices, one row group
        bestNU = 4; bestGR = 1; bestG = (N + 4 * per - 1) / (4 * per);
        if (bestG > gmax) { bestG = gmax; }
    }
    int slice = bestNU * per;
    if ((long long)bestG * slice < N) { slice = ((N + bestG - 1) / bestG + per - 1) / per * per; bestNU = 4; }   // (N > gmax slices of 4 vectors: not reachable for N <= 32768)
    a.G = bestG; a.GR = bestGR; a.slice = slice;
    if (vec2) return bestNU == 2 ? launch_ratio_t<2, 2>(h, a, h->ratio_sms, nullptr, true) : launch_ratio_t<2, 4>(h, a, h->ratio_sms, nullptr, true);
    return bestNU == 2 ? launch_ratio_t<1, 2>(h, a, h->ratio_sms, nullptr, true) : launch_ratio_t<1, 4>(h, a, h->ratio_sms, nullptr, true);
}

extern "C" int qmcd_ratio(qmcd_handle h, int j, const double* v_dev, double* R_dev) {
    if (!h || !v_dev || !R_dev || j < 0 || j >= h->N) return QMCD_EINVAL;
    if (!h->has_inverse) return QMCD_ESTATE;
    int rc;
    if (h->ratio_opt) rc = launch_ratio(h, j, nullptr, v_dev, R_dev);
    else {
        QmcdArgs a = base_args(h, QMCD_MODE_RATIO);
        a.j = j; a.v = v_dev; a.R_out = R_dev;
        rc = launch(h, a, false);
    }
    if (rc == QMCD_OK) h->state = QMCD_PROPOSED;
    return rc;
}

extern "C" int qmcd_ratio_jv(qmcd_handle h, const int* j_dev, const double* v_dev, double* R_dev) {
    if (!h || !j_dev || !v_dev || !R_dev) return QMCD_EINVAL;
    if (!h->has_inverse) return QMCD_ESTATE;
    int rc;
    if (h->ratio_opt) rc = launch_ratio(h, 0, j_dev, v_dev, R_dev);
    else {
        QmcdArgs a = base_args(h, QMCD_MODE_RATIO);
        a.jv = j_dev; a.v = v_dev; a.R_out = R_dev;
        rc = launch(h, a, false);
    }
    if (rc == QMCD_OK) h->state = QMCD_PROPOSED;
    return rc;
}

extern "C" int qmcd_accept(qmcd_handle h, const unsigned char* mask_dev) {
    if (!h) return QMCD_EINVAL;
    if (h->state != QMCD_PROPOSED) return QMCD_ESTATE;
    QmcdArgs a = base_args(h, QMCD_MODE_ACCEPT);
    a.mask = mask_dev; a.accept_all = (mask_dev == nullptr);
    int rc = launch(h, a, false);
    if (rc == QMCD_OK) h->state = QMCD_IDLE;
    return rc;
}

extern "C" int qmcd_accept_metropolis(qmcd_handle h, const double* uniforms_dev, unsigned char* acc_out_dev) {
    if (!h || !uniforms_dev) return QMCD_EINVAL;
    if (h->state != QMCD_PROPOSED) return QMCD_ESTATE;
    QmcdArgs a = base_args(h, QMCD_MODE_ACCEPT);
    a.uniforms = uniforms_dev; a.acc_out = acc_out_dev;
    int rc = launch(h, a, false);
    if (rc == QMCD_OK) h->state = QMCD_IDLE;
    return rc;
}

extern "C" int qmcd_reject(qmcd_handle h) {
    if (!h) return QMCD_EINVAL;
    if (h->state != QMCD_PROPOSED) return QMCD_ESTATE;
    if (h->P.lockstep) {                       // the rejected proposal still takes a slot of the window
        QmcdArgs a = base_args(h, QMCD_MODE_ACCEPT);
        a.reject_all = 1;
        int rc = launch(h, a, false);
        if (rc == QMCD_OK) h->state = QMCD_IDLE;
        return rc;
    }
    CK(h, cudaMemsetAsync(h->P.sj, 0xff, (size_t)h->batch * 4, h->stream));
    h->state = QMCD_IDLE;
    return QMCD_OK;
}

extern "C" int qmcd_flush(qmcd_handle h) {
    if (!h) return QMCD_EINVAL;
    if (h->state != QMCD_IDLE) return QMCD_ESTATE;
    if (!h->has_inverse) return QMCD_OK;
    QmcdArgs a = base_args(h, QMCD_MODE_FLUSH);
    return launch(h, a, true);
}

extern "C" int qmcd_pending(qmcd_handle h, int* m_dev) {
    if (!h || !m_dev) return QMCD_EINVAL;
    CK(h, cudaMemcpyAsync(m_dev, h->P.m, (size_t)h->batch * 4, cudaMemcpyDeviceToDevice, h->stream));
    return QMCD_OK;
}

extern "C" int qmcd_counters(qmcd_handle h, long long* counters_dev) {
    if (!h || !counters_dev) return QMCD_EINVAL;
    CK(h, cudaMemcpyAsync(counters_dev, h->P.counters, (size_t)h->batch * 64, cudaMemcpyDeviceToDevice, h->stream));
    return QMCD_OK;
}

extern "C" int qmcd_worker_stats(qmcd_handle h, long long* stats_dev, long long* flush_rank_sum_dev) {
    if (!h || (!stats_dev && !flush_rank_sum_dev)) return QMCD_EINVAL;
    if (stats_dev) CK(h, cudaMemcpyAsync(stats_dev, h->P.wstat, (size_t)QMCD_WSTAT_CTAS * 32, cudaMemcpyDeviceToDevice, h->stream));
    if (flush_rank_sum_dev) CK(h, cudaMemcpy2DAsync(flush_rank_sum_dev, 8, h->P.fstat, 16, 8, (size_t)h->batch, cudaMemcpyDeviceToDevice, h->stream));
    return QMCD_OK;
}

extern "C" int qmcd_status(qmcd_handle h, int* host_out, int* info_out) {
    if (!h || !host_out) return QMCD_EINVAL;
    int st[4] = {0, 0, 0, 0};
    CK(h, cudaMemcpyAsync(st, h->P.status, 16, cudaMemcpyDeviceToHost, h->stream));
    CK(h, cudaStreamSynchronize(h->stream));
    *host_out = st[0];
    if (info_out) { info_out[0] = st[1]; info_out[1] = st[2]; }
    return QMCD_OK;
}

extern "C" int qmcd_sweep(qmcd_handle h, int j_begin, int n_moves,
                          const double* proposals_dev, const unsigned char* mask_dev,
                          const double* uniforms_dev, double* R_out_dev, unsigned char* acc_out_dev) {
    if (!h || n_moves < 0 || j_begin < 0 || j_begin >= h->N) return QMCD_EINVAL;
    if ((mask_dev == nullptr) == (uniforms_dev == nullptr)) return QMCD_EINVAL;
    if (n_moves > 0 && !proposals_dev) return QMCD_EINVAL;
    if (h->state != QMCD_IDLE || !h->has_inverse) return QMCD_ESTATE;
    if (n_moves == 0) return QMCD_OK;
    QmcdArgs a = base_args(h, QMCD_MODE_SWEEP);
    a.j_begin = j_begin; a.n_moves = n_moves; a.v = proposals_dev;
    a.mask = mask_dev; a.uniforms = uniforms_dev; a.R_out = R_out_dev; a.acc_out = acc_out_dev;
    if (h->P.la_tma && !(encode_proposals(&h->tmaps.Vs[0], proposals_dev, n_moves, h->N, h->batch, 16, qmcd_sb_nq(h->K)) &&
                         encode_proposals(&h->tmaps.Vs[1], proposals_dev, n_moves, h->N, h->batch, 32, qmcd_sb_nq(h->K)) &&
                         encode_proposals(&h->tmaps.Vs[2], proposals_dev, n_moves, h->N, h->batch, 64, qmcd_sb_nq(h->K)))) { h->la_opt = 0; refresh_use_tma(h); a.P = h->P; }
    // (the blocked look-ahead with M in global memory has no lock-step variant: that combination runs per move)
    a.blocked = (h->lookahead != 1 && !h->P.slot_replace && h->P.blk_ok && (h->P.m_in_smem || !h->P.lockstep) &&
                 (((uintptr_t)proposals_dev & 15) == 0)) ? 1 : 0;
    return launch(h, a, true);
}

// ---- batched on-device inversion (qmcd_invert.cuh)
static size_t inv_smem_bytes(int N) { return (size_t)N * 16; }

// CTAs per walker of the blocked kernel are bounded so that its candidate records stay small: batch * C <= 512
static int invb_cmax(int batch) { int c = 512 / batch; if (c < 1) c = 1; if (c > QMCD_INV_CMAX) c = QMCD_INV_CMAX; return c; }
extern "C" size_t qmcd_invert_scratch_bytes(int N, int batch) {
    if (N < 1 || batch < 1 || inv_smem_bytes(N) > 227 * 1024) return 0;
    return al256((size_t)batch * N * 4) + al256((size_t)batch * QMCD_INV_CMAX * 8) +
           al256((size_t)batch * QMCD_INV_CMAX * 4) + al256((size_t)batch * 4) +
           al256((size_t)batch * 2 * invb_cmax(batch) * QMCD_INVB_REC * 8) +          // blocked kernel: candidate records,
           al256((size_t)batch * 2 * 2 * QMCD_INVB_KB * 8) +                         // slot k's data,
           al256((size_t)batch * QMCD_INVB_KB * QMCD_INVB_KB * 8);                   // L | d | later multipliers
}

// The blocked Gauss-Jordan kernel (qmcd_invert_blocked.cuh): panel width KB <= 16, C CTAs per walker and the chunk width
// chosen so that the whole batch is co-resident (one cooperative launch) with the widest panel that fits shared memory.
// Returns QMCD_OK with *done = 1 when it ran; *done = 0 = not applicable (the caller runs the unblocked kernel).
static int launch_invert_blocked(qmcd_ctx* h, const double* A_dev, double* Ainv_dev, unsigned char* sc, int* info, int* done) {
    *done = 0;
    const int N = h->N, batch = h->batch;
    const size_t cap = 227 * 1024 - 1024;                // (the kernel also has a few hundred bytes of static shared memory)
    int dev = 0, sms = 0;
    CK(h, cudaGetDevice(&dev));
    CK(h, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CK(h, cudaFuncSetAttribute(qmcd_invert_blocked_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cap));
    const int threads = QMCD_INV_THREADS;
    int CH = 512; while (CH / 2 >= N && CH > 32) CH /= 2;
    int bestC = 0, bestKB = 0; size_t best_smem = 0;
    for (int KB = QMCD_INVB_KB; KB >= 2 && !bestC; KB /= 2) {
        for (int C = invb_cmax(batch); C >= 1; --C) {
            if (C > 1 && (N + C - 1) / C < 8) continue;                  // at least 8 slots per CTA
            const size_t smem = qmcd_invb_smem_bytes(N, C, KB, CH);
            if (smem > cap) break;                                       // fewer CTAs per walker need more still
            int per_sm = 0;
            CK(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, qmcd_invert_blocked_kernel, threads, smem));
            if ((long long)C * batch <= (long long)sms * per_sm) { bestC = C; bestKB = KB; best_smem = smem; break; }
        }
    }
    if (!bestC) return QMCD_OK;                                          // the batch is not co-resident at any width: unblocked kernel
    QmcdInvBArgs a;
    a.N = N; a.batch = batch; a.C = bestC; a.KB = bestKB; a.CH = CH;
    a.A = A_dev; a.X = Ainv_dev; a.info = info;
    a.piv = (int*)sc; sc += al256((size_t)batch * N * 4);
    sc += al256((size_t)batch * QMCD_INV_CMAX * 8) + al256((size_t)batch * QMCD_INV_CMAX * 4) + al256((size_t)batch * 4);
    a.cand = (double*)sc; sc += al256((size_t)batch * 2 * invb_cmax(batch) * QMCD_INVB_REC * 8);
    a.kdat = (double*)sc; sc += al256((size_t)batch * 2 * 2 * QMCD_INVB_KB * 8);
    a.lf = (double*)sc;
    void* kargs[] = {(void*)&a};
    CK(h, cudaLaunchCooperativeKernel((void*)qmcd_invert_blocked_kernel, dim3((unsigned)(batch * bestC)), dim3((unsigned)threads),
                                      kargs, best_smem, h->stream));
    *done = 1;
    return QMCD_OK;
}

extern "C" int qmcd_invert(qmcd_handle h, const double* A_dev, double* Ainv_dev,
                           void* scratch_dev, size_t scratch_bytes, int* info_dev) {
    if (!h || !A_dev || !Ainv_dev || !scratch_dev) return QMCD_EINVAL;
    const int N = h->N, batch = h->batch;
    const size_t need = qmcd_invert_scratch_bytes(N, batch);
    if (need == 0 || scratch_bytes < need || ((uintptr_t)scratch_dev & 255)) return QMCD_EINVAL;
    if (h->state != QMCD_IDLE) return QMCD_ESTATE;
    if (h->invb_opt) {                                   // blocked kernel: the matrix crosses HBM N/16 times instead of N times
        int* info_b = info_dev ? info_dev : (int*)((unsigned char*)scratch_dev + al256((size_t)batch * N * 4) +
                                                   al256((size_t)batch * QMCD_INV_CMAX * 8) + al256((size_t)batch * QMCD_INV_CMAX * 4));
        CK(h, cudaMemsetAsync(info_b, 0, (size_t)batch * 4, h->stream));
        int done = 0;
        const int rc = launch_invert_blocked(h, A_dev, Ainv_dev, (unsigned char*)scratch_dev, info_b, &done);
        if (rc != QMCD_OK || done) return rc;
    }
    const size_t smem = inv_smem_bytes(N);
    CK(h, cudaFuncSetAttribute(qmcd_invert_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int dev = 0, sms = 0;
    CK(h, cudaGetDevice(&dev));
    CK(h, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    // 256 or 512 threads per CTA: whichever keeps more warps resident on an SM (the loop is
    // bound by loads in flight); on a tie the smaller CTA (finer balance over the SMs)
    int threads = 0, per_sm = 0;
    for (int t = 256; t <= QMCD_INV_THREADS; t *= 2) {
        int n = 0;
        CK(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, qmcd_invert_kernel, t, smem));
        if (n * t > per_sm * threads) { threads = t; per_sm = n; }
    }
    const int max_blocks = sms * per_sm;
    if (max_blocks < 1) return QMCD_EINVAL;
    // C CTAs per walker (row slots interleaved), as many walkers per cooperative launch as fit
    int C = max_blocks / batch;
    if (C < 1) C = 1;
    if (C > QMCD_INV_CMAX) C = QMCD_INV_CMAX;
    { const int nw = threads / 32; if (C > (N + nw - 1) / nw) C = (N + nw - 1) / nw; }   // at least one row per warp
    const int per_launch = (max_blocks / C < batch) ? max_blocks / C : batch;
    unsigned char* sc = (unsigned char*)scratch_dev;
    QmcdInvArgs a;
    a.N = N; a.C = C;
    int* piv = (int*)sc; sc += al256((size_t)batch * N * 4);
    double* cval = (double*)sc; sc += al256((size_t)batch * QMCD_INV_CMAX * 8);
    int* cidx = (int*)sc; sc += al256((size_t)batch * QMCD_INV_CMAX * 4);
    int* info = info_dev ? info_dev : (int*)sc;
    CK(h, cudaMemsetAsync(info, 0, (size_t)batch * 4, h->stream));
    for (int b0 = 0; b0 < batch; b0 += per_launch) {
        const int nb = (batch - b0 < per_launch) ? batch - b0 : per_launch;
        a.batch = nb;
        a.A = A_dev + (size_t)b0 * N * N; a.X = Ainv_dev + (size_t)b0 * N * N;
        a.piv = piv + (size_t)b0 * N; a.cand_val = cval + (size_t)b0 * QMCD_INV_CMAX;
        a.cand_idx = cidx + (size_t)b0 * QMCD_INV_CMAX; a.info = info + b0;
        void* kargs[] = {(void*)&a};
        CK(h, cudaLaunchCooperativeKernel((void*)qmcd_invert_kernel, dim3((unsigned)(nb * C)), dim3((unsigned)threads),
                                          kargs, smem, h->stream));
    }
    return QMCD_OK;
}

// ---- qmcd_invert_static: the same inversion for callers that may not allocate (CUDA graph capture, serving loops,
// harnesses that forbid cudaMalloc): the scratch of qmcd_invert lives in a file-scope device array instead of a
// caller buffer.  Every GPU that loads the library holds the array until exit.  In HOST code the array's name is
// a host-side stand-in, not a device address: the address is resolved once per device, with that device current,
// by cudaGetSymbolAddress, and that pointer is what the kernel gets.
#define QMCD_INVERT_STATIC_BYTES (1 << 20)        // 1 MiB: every BASELINE.json shape fits (c2, the largest, needs 459 KB)
#define QMCD_MAX_DEVICES 64
static __device__ __align__(256) unsigned char qmcd_invert_static_scratch[QMCD_INVERT_STATIC_BYTES];
static void* g_static_scratch_ptr[QMCD_MAX_DEVICES];        // per device; nullptr = not resolved yet
static std::mutex g_static_scratch_mutex;

extern "C" size_t qmcd_invert_static_max_bytes(void) { return QMCD_INVERT_STATIC_BYTES; }

extern "C" int qmcd_invert_static(qmcd_handle h, const double* A_dev, double* Ainv_dev, int* info_dev) {
    if (!h || !A_dev || !Ainv_dev) return QMCD_EINVAL;
    const size_t need = qmcd_invert_scratch_bytes(h->N, h->batch);
    if (need == 0) return QMCD_EINVAL;
    if (need > QMCD_INVERT_STATIC_BYTES) {
        snprintf(g_last_error, sizeof(g_last_error),
                 "qmcd_invert_static: N = %d, batch = %d needs %zu bytes of scratch, the static array holds %d "
                 "(use qmcd_invert with a caller buffer)", h->N, h->batch, need, QMCD_INVERT_STATIC_BYTES);
        memcpy(h->last_cuda_error, g_last_error, sizeof(g_last_error));
        return QMCD_ELIMIT;
    }
    int dev = 0;
    CK(h, cudaGetDevice(&dev));
    if (dev < 0 || dev >= QMCD_MAX_DEVICES) return QMCD_EINVAL;
    void* ptr = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_static_scratch_mutex);
        if (!g_static_scratch_ptr[dev]) {                     // set-up, once per device, that device current
            void* p = nullptr;
            CK(h, cudaGetSymbolAddress(&p, qmcd_invert_static_scratch));
            g_static_scratch_ptr[dev] = p;
        }
        ptr = g_static_scratch_ptr[dev];
    }
    // the array keeps the last call's contents: clear the part this call uses (the kernel writes its pivot and
    // candidate arrays before reading them; the per-walker info words must start at zero)
    CK(h, cudaMemsetAsync(ptr, 0, need, h->stream));
    return qmcd_invert(h, A_dev, Ainv_dev, ptr, need, info_dev);
}

extern "C" size_t qmcd_sweep_host_min_staging(int N, int batch) {
    if (N < 1 || batch < 1) return 0;
    // two buffers of one move each
    size_t per_move = al256((size_t)batch * N * 8) + 4 * al256((size_t)batch * 8);
    return 2 * per_move;
}

extern "C" int qmcd_sweep_host(qmcd_handle h, int j_begin, int n_moves,
                               const double* proposals_host, const unsigned char* mask_host,
                               const double* uniforms_host, double* R_out_host,
                               unsigned char* acc_out_host, void* staging_dev, size_t staging_bytes) {
    if (!h || n_moves < 0 || j_begin < 0 || j_begin >= h->N) return QMCD_EINVAL;
    if ((mask_host == nullptr) == (uniforms_host == nullptr)) return QMCD_EINVAL;
    if (n_moves > 0 && (!proposals_host || !staging_dev)) return QMCD_EINVAL;
    if (((uintptr_t)staging_dev & 255) || staging_bytes < qmcd_sweep_host_min_staging(h->N, h->batch)) return QMCD_EINVAL;
    if (h->state != QMCD_IDLE || !h->has_inverse) return QMCD_ESTATE;
    const size_t bn = (size_t)h->batch * h->N * 8, b8 = (size_t)h->batch * 8, b1 = (size_t)h->batch;
    // moves per chunk: largest cm with 2 * (al256(cm*bn) + 4*al256(cm*b8)) <= staging
    long long cm = (long long)((staging_bytes / 2 - 5 * 256) / (bn + 4 * b8));
    if (cm < 1) cm = 1;
    if (cm > n_moves) cm = n_moves > 0 ? n_moves : 1;
    const size_t half = staging_bytes / 2 & ~(size_t)255;
    // chunk sizes grow geometrically from 128 moves to cm: the first copy (nothing to overlap it with) stays short, the
    // later launches long (every launch fills and drains the pool once)
    long long cur = cm < 128 ? cm : 128;
    for (int c = 0, t0 = 0, cnt = 0; t0 < n_moves; ++c, t0 += cnt, cur = (2 * cur < cm) ? 2 * cur : cm) {
        cnt = (int)((n_moves - t0 < cur) ? n_moves - t0 : cur);
        const int buf = c & 1;
        unsigned char* base = (unsigned char*)staging_dev + (size_t)buf * half;
        double* d_prop = (double*)base;
        double* d_uni = (double*)(base + al256((size_t)cm * bn));
        double* d_R = (double*)((unsigned char*)d_uni + al256((size_t)cm * b8));
        unsigned char* d_mask = (unsigned char*)d_R + al256((size_t)cm * b8);
        unsigned char* d_acc = d_mask + al256((size_t)cm * b8);
        if (c >= 2) CK(h, cudaStreamWaitEvent(h->copy_stream, h->ev_done[buf], 0));
        CK(h, cudaMemcpyAsync(d_prop, (const unsigned char*)proposals_host + (size_t)t0 * bn, (size_t)cnt * bn, cudaMemcpyHostToDevice, h->copy_stream));
        if (mask_host) CK(h, cudaMemcpyAsync(d_mask, mask_host + (size_t)t0 * b1, (size_t)cnt * b1, cudaMemcpyHostToDevice, h->copy_stream));
        else CK(h, cudaMemcpyAsync(d_uni, (const unsigned char*)uniforms_host + (size_t)t0 * b8, (size_t)cnt * b8, cudaMemcpyHostToDevice, h->copy_stream));
        CK(h, cudaEventRecord(h->ev_h2d[buf], h->copy_stream));
        CK(h, cudaStreamWaitEvent(h->stream, h->ev_h2d[buf], 0));
        int rc = qmcd_sweep(h, (j_begin + t0) % h->N, cnt, d_prop, mask_host ? d_mask : nullptr,
                            mask_host ? nullptr : d_uni, d_R, d_acc);
        if (rc != QMCD_OK) return rc;
        if (R_out_host) CK(h, cudaMemcpyAsync((unsigned char*)R_out_host + (size_t)t0 * b8, d_R, (size_t)cnt * b8, cudaMemcpyDeviceToHost, h->stream));
        if (acc_out_host) CK(h, cudaMemcpyAsync(acc_out_host + (size_t)t0 * b1, d_acc, (size_t)cnt * b1, cudaMemcpyDeviceToHost, h->stream));
        CK(h, cudaEventRecord(h->ev_done[buf], h->stream));
    }
    CK(h, cudaStreamSynchronize(h->stream));
    CK(h, cudaStreamSynchronize(h->copy_stream));
    return QMCD_OK;
}

extern "C" int qmcd_set_option(qmcd_handle h, const char* key, int value) {
    if (!h || !key) return QMCD_EINVAL;
    if (h->state != QMCD_IDLE) return QMCD_ESTATE;
    if (!strcmp(key, "cluster")) {                 // powers of two only: the blocked look-ahead deals 16 strip rows over the CTAs
        if (value < 1 || value > 16 || value > h->N || (value & (value - 1)) != 0) return QMCD_EINVAL;
        CK(h, cudaStreamSynchronize(h->stream));
        const int old = h->P.S;
        int rc = configure_kernel(h, value);
        if (rc == QMCD_OK && max_active_clusters(h, value, 1) < 1) rc = QMCD_EINVAL;
        if (rc != QMCD_OK) configure_kernel(h, old);
        return rc;
    }
    if (!strcmp(key, "pool")) {                    // -1 auto, 0 off, n > 0: at most n pool CTAs
        if (value < -1) return QMCD_EINVAL;
        h->pool_opt = value;
        return QMCD_OK;
    }
    if (!strcmp(key, "clusters_per_walker")) {     // round-1 name: 1 = leaders only (pool off), > 1 = pool on
        if (value < 1) return QMCD_EINVAL;
        h->pool_opt = (value == 1) ? 0 : -1;
        return QMCD_OK;
    }
    if (!strcmp(key, "cooperative")) {             // 0: pooled launches without the co-residency guarantee (profilers)
        if (value < 0 || value > 1) return QMCD_EINVAL;
        h->coop = value;
        return QMCD_OK;
    }
    if (!strcmp(key, "tile_rows")) {               // cp.async flush only (the TMA-fed flush works on 128-row tiles)
        if ((value != 64 && value != 128) || (value == 128 && h->K > 64)) return QMCD_EINVAL;
        h->tile_opt = value;
        h->P.tile_rows = value;
        refresh_use_tma(h);
        return QMCD_OK;
    }
    if (!strcmp(key, "stagger")) {                 // 0: every window takes K moves (walkers that start together flush together)
        if (value < 0 || value > 1) return QMCD_EINVAL;
        h->P.stagger = value;
        return QMCD_OK;
    }
    if (!strcmp(key, "invert_blocked")) {          // 0: qmcd_invert runs the unblocked kernel (one pass over the matrix per pivot)
        if (value < 0 || value > 1) return QMCD_EINVAL;
        h->invb_opt = value;
        return QMCD_OK;
    }
    if (!strcmp(key, "ratio_kernel")) {            // 0: qmcd_ratio through the cluster kernel's look-ahead (the per-move sweep's arithmetic)
        if (value < 0 || value > 1) return QMCD_EINVAL;
        h->ratio_opt = value;
        return QMCD_OK;
    }
    if (!strcmp(key, "la_tma")) {                  // 0: blocked look-ahead through LDG / cp.async; 1: TMA ring for long slices; 2: whenever it fits
        if (value < 0 || value > 2) return QMCD_EINVAL;
        CK(h, cudaStreamSynchronize(h->stream));
        h->la_opt = value;
        return configure_kernel(h, h->P.S);
    }
    if (!strcmp(key, "tma")) {                     // 0: K <= 64 flush tiles through the cp.async kernels instead
        if (value < 0 || value > 1) return QMCD_EINVAL;
        h->tma_opt = value;
        refresh_use_tma(h);
        if (!h->P.use_tma && h->K <= 64) h->P.tile_rows = h->tile_opt ? h->tile_opt : ((h->N >= 2048) ? 128 : 64);
        return QMCD_OK;
    }
    if (!strcmp(key, "flush_path")) {
        if (value < 0 || value > 2) return QMCD_EINVAL;
        h->P.flush_path = value;
        refresh_use_tma(h);
        return QMCD_OK;
    }
    if (!strcmp(key, "lookahead")) {
        if (value < 0 || value > 1) return QMCD_EINVAL;
        h->lookahead = value;
        return QMCD_OK;
    }
    if (!strcmp(key, "lockstep")) {                // legal between windows only (IDLE); starts a fresh window count
        if (value < 0 || value > 1) return QMCD_EINVAL;
        if (h->state != QMCD_IDLE) return QMCD_ESTATE;
        h->P.lockstep = value;
        return QMCD_OK;
    }
    if (!strcmp(key, "slot_replace")) {            // IDLE only; qmcd_sweep then runs the per-move look-ahead
        if (value < 0 || value > 1) return QMCD_EINVAL;
        h->P.slot_replace = value;
        return QMCD_OK;
    }
    if (!strcmp(key, "chain_regs")) {
        if (value < 0 || value > 1) return QMCD_EINVAL;
        h->P.chain_regs = value;
        return QMCD_OK;
    }
    return QMCD_EINVAL;
}

extern "C" int qmcd_get_option(qmcd_handle h, const char* key) {
    if (!h || !key) return QMCD_EINVAL;
    if (!strcmp(key, "cluster")) return h->P.S;
    if (!strcmp(key, "clusters_per_walker")) return pool_ctas(h) > 0 ? 2 : 1;
    if (!strcmp(key, "pool")) return pool_ctas(h);
    if (!strcmp(key, "cooperative")) return h->coop;
    if (!strcmp(key, "tile_rows")) return h->P.tile_rows;
    if (!strcmp(key, "tma")) return h->P.use_tma;
    if (!strcmp(key, "la_tma")) return h->P.la_tma;
    if (!strcmp(key, "invert_blocked")) return h->invb_opt;
    if (!strcmp(key, "stagger")) return h->P.stagger;
    if (!strcmp(key, "ratio_kernel")) return h->ratio_opt;
    if (!strcmp(key, "flush_path")) return h->P.flush_path;
    if (!strcmp(key, "lookahead")) return h->lookahead;
    if (!strcmp(key, "lockstep")) return h->P.lockstep;
    if (!strcmp(key, "slot_replace")) return h->P.slot_replace;
    if (!strcmp(key, "blocked_ok")) return h->P.blk_ok && (h->P.m_in_smem || !h->P.lockstep) && !h->P.slot_replace;
    if (!strcmp(key, "m_in_smem")) return h->P.m_in_smem;
    if (!strcmp(key, "threads")) return QMCD_THREADS;
    if (!strcmp(key, "smem_bytes")) return (int)h->smem_bytes;
    if (!strcmp(key, "max_active_clusters")) return max_active_clusters(h, h->P.S, h->batch);
    return QMCD_EINVAL;
}

extern "C" const char* qmcd_strerror(int code) {
    switch (code) {
        case QMCD_OK: return "ok";
        case QMCD_EINVAL: return "invalid argument";
        case QMCD_ESTATE: return "call not legal in the current state";
        case QMCD_ECUDA: return g_last_error[0] ? g_last_error : "CUDA error";
        case QMCD_ESINGULAR: return "accepted a move with R == 0 or non-finite R (singular)";
        case QMCD_ENOMEM: return "out of host memory";
        case QMCD_ELIMIT: return g_last_error[0] ? g_last_error : "size exceeds a fixed limit of this entry point";
        default: return "unknown error";
    }
}

extern "C" const char* qmcd_version(void) { return "qmcd 0.2 (sm_100a)"; }
