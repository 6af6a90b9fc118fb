// qmcd_flush_mma.cuh -- FP64 tensor-core (DMMA) flush of Eq. 4, per tile of
// 128 / 64 rows of B (tiles are taken one at a time by whichever CTA is free: qmcd_kernel.cuh):
//     T = B0 C^T - E_J   (row tile x m, reduction over N)          "NT stage"
//     K <= 64:  T <- T M (warp-local)                              "TM stage"
//               B <- B0 - T W                                      "NN stage"
//     K >  64:  Y = M W first (m x N, a job of 64-column tiles of its own), then B <- B0 - T Y
// sm_100a has no tcgen05 f64 kind; its FP64 tensor instruction is DMMA.8x8x4
// (mma.sync.m8n8k4.f64), measured at 37 TFLOP/s against 34 for DFMA.  Operand
// fragments are loaded as 16-byte vectors by permuting the contraction index
// (k-slot c of k-step s is k = 8q + 2c + s on BOTH operands) and, in the NN
// stage, the output columns (n-slot g of tile t is column 16G + 2g + t), which
// also makes every global access of B a full 128-byte line per 4 lanes.
#pragma once
#include "qmcd_phases.cuh"

#define QMCD_MMA_KC 64          // chunk extent (doubles) of every staged operand
#define QMCD_MMA_LDC 72         // NT-stage chunk row stride: == 8 (mod 16) doubles
#define QMCD_MMA_LDX 66         // NN-stage chunk row stride: == 2 (mod 8) doubles
#define QMCD_MMA_CHUNK_DOUBLES (64 * QMCD_MMA_LDC)

__host__ __device__ inline int qmcd_mma_ldT(int K) { return ((K + 15) / 16) * 16 + 8; }
// rows per tile: 128 (16 per warp) while T fits beside the two chunk buffers, else 64
__host__ __device__ inline int qmcd_mma_rows(int K) { return (K <= 64) ? 128 : 64; }
// operand chunks in flight: 3 (prefetch two chunks ahead) while they fit, else 2
__host__ __device__ inline int qmcd_mma_stages(int K) { return (K <= 128) ? 3 : 2; }
__host__ __device__ inline size_t qmcd_flush_mma_smem_bytes(int N, int K) {
    (void)N;
    return (size_t)qmcd_mma_rows(K) * qmcd_mma_ldT(K) * 8 + qmcd_mma_stages(K) * (size_t)QMCD_MMA_CHUNK_DOUBLES * 8 +
           (K <= 64 ? (size_t)64 * QMCD_MMA_LDX * 8 : 0);      // + M for the local T M stage
}

__device__ __forceinline__ void qmcd_dmma(double& d0, double& d1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
__device__ __forceinline__ void qmcd_cp_async16(void* smem_dst, const void* gsrc) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void qmcd_cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N_> __device__ __forceinline__ void qmcd_cp_async_wait() {
    asm volatile("cp.async.wait_group %0;" :: "n"(N_) : "memory");
}

__device__ inline bool qmcd_flush_use_mma(const QmcdDev& P) {
    if (P.flush_path == 1) return false;
    // rank 1 (the K = 1 Sherman-Morrison path) too: measured 2-4x faster than the CUDA-core flush
    return (P.N % 64 == 0) && P.mma_smem_ok;
}

// Stage `nrows` (<= 64, multiple of 8 after zero padding) rows x 64 columns of a
// row-major [m][ld] global matrix into a chunk buffer with row stride LD.
// Rows >= m_valid are zero-filled.  All 256 threads; caller commits / waits.
template <int LD>
__device__ __forceinline__ void qmcd_stage_chunk(double* __restrict__ dst, const double* __restrict__ src,
                                                 size_t ld, int row0, int nrows, int m_valid, int col0) {
    const int tid = threadIdx.x;
    // 64 columns = 32 x 16 B per row
    for (int idx = tid; idx < nrows * 32; idx += QMCD_THREADS) {
        const int i = idx >> 5, c2 = (idx & 31) * 2;
        double* d = dst + i * LD + c2;
        if (row0 + i < m_valid) qmcd_cp_async16(d, src + (size_t)(row0 + i) * ld + col0 + c2);
        else { d[0] = 0.0; d[1] = 0.0; }
    }
}

// Same, but only the warps of group `half` (warps 4*half .. 4*half+3) stage, and only rows
// [32*half, 32*half + 32): the two warps that share a scheduler stage at different
// times (start / middle of a chunk's MMAs), so one's copies overlap the other's MMAs.
template <int LD>
__device__ __forceinline__ void qmcd_stage_half(double* __restrict__ dst, const double* __restrict__ src,
                                                size_t ld, int row0, int nrows, int m_valid, int col0, int half) {
    const int t = threadIdx.x & 127;
    const int rlo = 32 * half, rhi = min(nrows, rlo + 32);
    for (int idx = rlo * 32 + t; idx < rhi * 32; idx += 128) {
        const int i = idx >> 5, c2 = (idx & 31) * 2;
        double* d = dst + i * LD + c2;
        if (row0 + i < m_valid) qmcd_cp_async16(d, src + (size_t)(row0 + i) * ld + col0 + c2);
        else { d[0] = 0.0; d[1] = 0.0; }
    }
}

__device__ __forceinline__ double2 qmcd_lds128(const double* p) { return *reinterpret_cast<const double2*>(p); }
// the same from a 32-bit shared-memory address: LDS.128 whatever the compiler knows about the pointer's origin (a generic
// pointer that reaches a __noinline__ function is read with LD.E.128 plus descriptor moves)
__device__ __forceinline__ double2 qmcd_lds128s(unsigned a) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ double qmcd_lds64s(unsigned a) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a) : "memory");
    return v;
}
// coherent 16-byte global load / store of B: the same kernel rewrites B, and a tile is taken by a
// different CTA from one flush to the next, so the loads go to L2 (.cg), never through L1
__device__ __forceinline__ double2 qmcd_ldg128(const double* p) {
    double2 v;
    asm volatile("ld.global.cg.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void qmcd_stg128(double* p, double x, double y) {
    asm volatile("st.global.v2.f64 [%0], {%1,%2};" :: "l"(p), "d"(x), "d"(y) : "memory");
}

// ---------------------------------------------------------------------------
// NT stage:  Ts[r][i] = -( sum_k B[row0+r][k] C[i][k] ) + delta(row0+r, J[i])
// for the R = 64*A_T rows of one tile and all i < m (zero for m <= i < mp8).
// Warp w owns tile rows [8 A_T w, 8 A_T (w+1)); its A fragments come straight
// from global memory (16 B per lane, prefetched one k-group ahead), the C chunk
// is staged once per CTA with cp.async and shared by the 8 warps.
// ---------------------------------------------------------------------------
template <int A_T, int NB, int NS>
__device__ void qmcd_mma_nt(const double* Bw, int N, int row0, int nvalid,
                            const double* __restrict__ Cq, const int* __restrict__ Jq, int m,
                            double* __restrict__ Ts, int ldT, double* __restrict__ cb) {
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, g = lane >> 2, c = lane & 3;
    const int mp8 = (m + 7) & ~7;
    const int nchunks = N / QMCD_MMA_KC;
    const double* ap[A_T];
    bool av[A_T];
#pragma unroll
    for (int a = 0; a < A_T; ++a) {
        const int r = wid * 8 * A_T + a * 8 + g;
        av[a] = r < nvalid;
        ap[a] = Bw + (size_t)(row0 + (av[a] ? r : 0)) * N + 2 * c;
    }
    // T is produced NB*8 columns at a time (rows of C past m are staged as zeros)
    for (int col0 = 0; col0 < mp8; col0 += NB * 8) {
        constexpr int ncols = NB * 8;
        double acc[A_T][NB][2];
#pragma unroll
        for (int a = 0; a < A_T; ++a)
#pragma unroll
            for (int b = 0; b < NB; ++b) { acc[a][b][0] = 0.0; acc[a][b][1] = 0.0; }
        __syncthreads();                         // every warp is done with the chunk buffers
#pragma unroll
        for (int i = 0; i < NS - 1; ++i) {
            if (i < nchunks) qmcd_stage_chunk<QMCD_MMA_LDC>(cb + i * QMCD_MMA_CHUNK_DOUBLES, Cq, (size_t)N, col0, ncols, m, i * QMCD_MMA_KC);
            qmcd_cp_async_commit();
        }
        // A fragments: a ring of 4 k-groups (32 columns) ahead of the MMAs
        double2 ar[4][A_T];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int a = 0; a < A_T; ++a) ar[i][a] = av[a] ? qmcd_ldg128(ap[a] + 8 * i) : make_double2(0.0, 0.0);
        for (int kc = 0; kc < nchunks; ++kc) {
            qmcd_cp_async_wait<NS - 2>();
            __syncthreads();                     // chunk kc landed; buffer (kc-1)%NS is free
            const double* cur = cb + (kc % NS) * QMCD_MMA_CHUNK_DOUBLES + g * QMCD_MMA_LDC + 2 * c;
            double2 bn[NB];                      // C fragments of k-group q+1, loaded during k-group q
#pragma unroll
            for (int b = 0; b < NB; ++b) bn[b] = qmcd_lds128(cur + b * 8 * QMCD_MMA_LDC);
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                if (q == 4 * (wid >> 2)) {       // warps 0-3 stage at q = 0, warps 4-7 at q = 4
                    if (kc + NS - 1 < nchunks)
                        qmcd_stage_half<QMCD_MMA_LDC>(cb + ((kc + NS - 1) % NS) * QMCD_MMA_CHUNK_DOUBLES, Cq, (size_t)N, col0,
                                                      ncols, m, (kc + NS - 1) * QMCD_MMA_KC, wid >> 2);
                    qmcd_cp_async_commit();
                }
                double2 a_cur[A_T];
#pragma unroll
                for (int a = 0; a < A_T; ++a) a_cur[a] = ar[q & 3][a];
                const int nk = kc * QMCD_MMA_KC + (q + 4) * 8;
                if (nk < N) {
#pragma unroll
                    for (int a = 0; a < A_T; ++a)
                        if (av[a]) ar[q & 3][a] = qmcd_ldg128(ap[a] + nk);
                }
                // all k-step-0 MMAs, then all k-step-1 MMAs: consecutive DMMAs are independent
                double2 bv[NB];
#pragma unroll
                for (int b = 0; b < NB; ++b) bv[b] = bn[b];
                if (q < 7) {
#pragma unroll
                    for (int b = 0; b < NB; ++b) bn[b] = qmcd_lds128(cur + b * 8 * QMCD_MMA_LDC + 8 * (q + 1));
                }
#pragma unroll
                for (int b = 0; b < NB; ++b)
#pragma unroll
                    for (int a = 0; a < A_T; ++a) qmcd_dmma(acc[a][b][0], acc[a][b][1], a_cur[a].x, bv[b].x);
#pragma unroll
                for (int b = 0; b < NB; ++b)
#pragma unroll
                    for (int a = 0; a < A_T; ++a) qmcd_dmma(acc[a][b][0], acc[a][b][1], a_cur[a].y, bv[b].y);
            }
        }
        qmcd_cp_async_wait<0>();
#pragma unroll
        for (int a = 0; a < A_T; ++a)
#pragma unroll
            for (int b = 0; b < NB; ++b)
                if (col0 + b * 8 < mp8)
                    *reinterpret_cast<double2*>(Ts + (size_t)(wid * 8 * A_T + a * 8 + g) * ldT + col0 + b * 8 + 2 * c) =
                        make_double2(-acc[a][b][0], -acc[a][b][1]);
    }
    __syncthreads();
    for (int i = tid; i < m; i += QMCD_THREADS) {
        const int r = __ldcg(Jq + i) - row0;
        if (r >= 0 && r < 64 * A_T) Ts[(size_t)r * ldT + i] += 1.0;
    }
    __syncthreads();
}

// ---------------------------------------------------------------------------
// NN stage:  D[row0+r][n] = (INIT ? D[row0+r][n] : 0) + sum_a Ts[r][a] X[a][n]
// for tile rows r < nvalid and columns n in [c_lo, c_hi) (multiple of 64 wide),
// a < kext (X rows >= m_valid read as zero).  X is staged in 64 x 64 chunks
// (cp.async ring of NS buffers, one __syncthreads per chunk).  A warp owns 8 A_T
// rows and works in PASSES of 64 / A_T columns (16 accumulator registers pairs):
// while pass p's MMAs run, the 8 vectors of pass p+1's initial D values are
// loaded and the 8 result vectors of pass p-1 are stored, one of each per
// k-group, so loads, MMAs and stores of three consecutive passes overlap and the
// store queue never sees a burst.  A_T = 2 needs kext <= 64 (one k-chunk).
// ---------------------------------------------------------------------------
template <int A_T, bool INIT, int NS>
__device__ void qmcd_mma_nn(const double* __restrict__ Ts, int ldT, int kext,
                            const double* __restrict__ X, int m_valid, int N,
                            double* D, int row0, int nvalid, int c_lo, int c_hi,
                            double* __restrict__ cb) {
    constexpr int GH = 4 / A_T;          // 16-column groups per pass
    constexpr int NP = A_T;              // passes per 64-column chunk
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, g = lane >> 2, c = lane & 3;
    const int nk = (kext + 63) >> 6;
    const int nn = (c_hi - c_lo) >> 6;
    const int total = nn * nk;
    const int npass = nn * NP;
    bool rv[A_T];
    double* dp[A_T];
    const double* tp[A_T];
#pragma unroll
    for (int a = 0; a < A_T; ++a) {
        const int r = wid * 8 * A_T + a * 8 + g;
        rv[a] = r < nvalid;
        dp[a] = D + (size_t)(row0 + (rv[a] ? r : 0)) * N + 4 * c;
        tp[a] = Ts + (size_t)r * ldT + 2 * c;
    }
    const bool warp_has_rows = wid * 8 * A_T < nvalid;       // warps without rows only help staging
    __syncthreads();                                         // every warp is done with the chunk buffers
#pragma unroll
    for (int i = 0; i < NS - 1; ++i) {
        if (i < total) {
            const int ni = i / nk, kb = i - ni * nk;
            qmcd_stage_chunk<QMCD_MMA_LDX>(cb + i * QMCD_MMA_CHUNK_DOUBLES, X, (size_t)N, kb * 64, min(64, kext - kb * 64),
                                           m_valid, c_lo + ni * 64);
        }
        qmcd_cp_async_commit();
    }
    // vector v = (a, Gl, h) of a pass: rows a, columns 16 (hp GH + Gl) + 4 c + 2 h .. +1
    double2 initn[8], outv[8];
#pragma unroll
    for (int v = 0; v < 8; ++v) {
        const int a = v / (2 * GH), Gl = (v >> 1) % GH, h = v & 1;
        initn[v] = (INIT && rv[a]) ? qmcd_ldg128(dp[a] + c_lo + 16 * Gl + 2 * h) : make_double2(0.0, 0.0);
        outv[v] = make_double2(0.0, 0.0);
    }
    int ci = 0, pprev_col = -1;
    for (int ni = 0; ni < nn; ++ni) {
        const int n0 = c_lo + ni * 64;
#pragma unroll
        for (int hp = 0; hp < NP; ++hp) {
            const int pcol = n0 + 16 * GH * hp;                       // first column of this pass
            const int pass = ni * NP + hp;
            const int ncol = (hp + 1 < NP) ? pcol + 16 * GH : n0 + 64; // first column of the next pass
            const bool has_next = pass + 1 < npass;
            double acc[A_T][GH][2][2];
#pragma unroll
            for (int a = 0; a < A_T; ++a)
#pragma unroll
                for (int Gl = 0; Gl < GH; ++Gl) {
                    const int v = (a * GH + Gl) * 2;
                    acc[a][Gl][0][0] = initn[v].x; acc[a][Gl][1][0] = initn[v].y;
                    acc[a][Gl][0][1] = initn[v + 1].x; acc[a][Gl][1][1] = initn[v + 1].y;
                }
            for (int kb = 0; kb < nk; ++kb) {
                if (hp == 0) {                   // a new chunk (with A_T = 2, nk == 1: both passes share it)
                    qmcd_cp_async_wait<NS - 2>();
                    __syncthreads();             // chunk ci landed; buffer (ci-1)%NS is free
                }
                const double* cur = cb + (ci % NS) * QMCD_MMA_CHUNK_DOUBLES + (2 * c) * QMCD_MMA_LDX + 2 * g + 16 * GH * hp;
                const int nq = min(64, kext - kb * 64) >> 3;
                double2 fa[A_T], f0[GH], f1[GH];
#pragma unroll
                for (int a = 0; a < A_T; ++a) fa[a] = qmcd_lds128(tp[a] + kb * 64);
#pragma unroll
                for (int Gl = 0; Gl < GH; ++Gl) {
                    f0[Gl] = qmcd_lds128(cur + 16 * Gl);
                    f1[Gl] = qmcd_lds128(cur + QMCD_MMA_LDX + 16 * Gl);
                }
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    // warps 0-3 stage at the chunk's first k-group, warps 4-7 half way through it
                    if ((wid < 4) ? (hp == 0 && q == 0) : (NP == 1 ? q == 4 : (hp == 1 && q == 0))) {
                        if (ci + NS - 1 < total) {
                            const int nci = ci + NS - 1, nni = nci / nk, nkb = nci - nni * nk;
                            qmcd_stage_half<QMCD_MMA_LDX>(cb + (nci % NS) * QMCD_MMA_CHUNK_DOUBLES, X, (size_t)N, nkb * 64,
                                                          min(64, kext - nkb * 64), m_valid, c_lo + nni * 64, wid >> 2);
                        }
                        qmcd_cp_async_commit();
                    }
                    if (kb == 0) {
                        // k-groups 0-3: the next pass's 8 initial vectors (two each, as early as
                        // possible); k-groups 4-7: the previous pass's 8 result vectors
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int v = 2 * (q & 3) + e;
                            const int a = v / (2 * GH), Gl = (v >> 1) % GH, h = v & 1;
                            if (rv[a]) {
                                if (q < 4) { if (INIT && has_next) initn[v] = qmcd_ldg128(dp[a] + ncol + 16 * Gl + 2 * h); }
                                else if (pprev_col >= 0) qmcd_stg128(dp[a] + pprev_col + 16 * Gl + 2 * h, outv[v].x, outv[v].y);
                            }
                        }
                    }
                    if (q < nq && warp_has_rows) {
                        // fragments of k-group q were loaded during k-group q-1
                        double2 avv[A_T], x0[GH], x1[GH];
#pragma unroll
                        for (int a = 0; a < A_T; ++a) avv[a] = fa[a];
#pragma unroll
                        for (int Gl = 0; Gl < GH; ++Gl) { x0[Gl] = f0[Gl]; x1[Gl] = f1[Gl]; }
                        if (q + 1 < nq) {
#pragma unroll
                            for (int a = 0; a < A_T; ++a) fa[a] = qmcd_lds128(tp[a] + kb * 64 + 8 * (q + 1));
#pragma unroll
                            for (int Gl = 0; Gl < GH; ++Gl) {
                                f0[Gl] = qmcd_lds128(cur + (8 * (q + 1)) * QMCD_MMA_LDX + 16 * Gl);
                                f1[Gl] = qmcd_lds128(cur + (8 * (q + 1) + 1) * QMCD_MMA_LDX + 16 * Gl);
                            }
                        }
#pragma unroll
                        for (int Gl = 0; Gl < GH; ++Gl)
#pragma unroll
                            for (int a = 0; a < A_T; ++a) {
                                qmcd_dmma(acc[a][Gl][0][0], acc[a][Gl][0][1], avv[a].x, x0[Gl].x);
                                qmcd_dmma(acc[a][Gl][1][0], acc[a][Gl][1][1], avv[a].x, x0[Gl].y);
                            }
#pragma unroll
                        for (int Gl = 0; Gl < GH; ++Gl)
#pragma unroll
                            for (int a = 0; a < A_T; ++a) {
                                qmcd_dmma(acc[a][Gl][0][0], acc[a][Gl][0][1], avv[a].y, x1[Gl].x);
                                qmcd_dmma(acc[a][Gl][1][0], acc[a][Gl][1][1], avv[a].y, x1[Gl].y);
                            }
                    }
                }
                if (hp == NP - 1) ++ci;
            }
#pragma unroll
            for (int a = 0; a < A_T; ++a)
#pragma unroll
                for (int Gl = 0; Gl < GH; ++Gl) {
                    const int v = (a * GH + Gl) * 2;
                    outv[v] = make_double2(acc[a][Gl][0][0], acc[a][Gl][1][0]);
                    outv[v + 1] = make_double2(acc[a][Gl][0][1], acc[a][Gl][1][1]);
                }
            pprev_col = pcol;
        }
    }
    if (pprev_col >= 0) {
#pragma unroll
        for (int v = 0; v < 8; ++v) {
            const int a = v / (2 * GH), Gl = (v >> 1) % GH, h = v & 1;
            if (rv[a]) qmcd_stg128(dp[a] + pprev_col + 16 * Gl + 2 * h, outv[v].x, outv[v].y);
        }
    }
    qmcd_cp_async_wait<0>();
}

// ---------------------------------------------------------------------------
// TM stage (m <= 64):  Ts <- Ts M  in place, warp-local (a warp owns its rows of Ts
// over all columns).  Mf: M staged in shared memory, [64][LDX], zero outside m x m.
// With it B <- B0 + Ts W needs neither Y = M W nor a barrier across the cluster.
// ---------------------------------------------------------------------------
template <int A_T>
__device__ void qmcd_mma_tm(double* __restrict__ Ts, int ldT, int mp8, const double* __restrict__ Mf) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, g = lane >> 2, c = lane & 3;
    const int nq = mp8 >> 3, nG = (mp8 + 15) >> 4;
    double* tp[A_T];
#pragma unroll
    for (int a = 0; a < A_T; ++a) tp[a] = Ts + (size_t)(wid * 8 * A_T + a * 8 + g) * ldT;
    double acc[A_T][4][2][2];
#pragma unroll
    for (int a = 0; a < A_T; ++a)
#pragma unroll
        for (int G = 0; G < 4; ++G) { acc[a][G][0][0] = acc[a][G][0][1] = acc[a][G][1][0] = acc[a][G][1][1] = 0.0; }
    const double* xb = Mf + (2 * c) * QMCD_MMA_LDX + 2 * g;
    for (int q = 0; q < nq; ++q) {
        double2 avv[A_T];
#pragma unroll
        for (int a = 0; a < A_T; ++a) avv[a] = qmcd_lds128(tp[a] + 2 * c + 8 * q);
#pragma unroll
        for (int G = 0; G < 4; ++G) {
            if (G < nG) {
                const double2 x0 = qmcd_lds128(xb + (8 * q) * QMCD_MMA_LDX + 16 * G);
                const double2 x1 = qmcd_lds128(xb + (8 * q + 1) * QMCD_MMA_LDX + 16 * G);
#pragma unroll
                for (int a = 0; a < A_T; ++a) {
                    qmcd_dmma(acc[a][G][0][0], acc[a][G][0][1], avv[a].x, x0.x);
                    qmcd_dmma(acc[a][G][1][0], acc[a][G][1][1], avv[a].x, x0.y);
                    qmcd_dmma(acc[a][G][0][0], acc[a][G][0][1], avv[a].y, x1.x);
                    qmcd_dmma(acc[a][G][1][0], acc[a][G][1][1], avv[a].y, x1.y);
                }
            }
        }
    }
    __syncwarp();                                    // all lanes have read this warp's rows of Ts
#pragma unroll
    for (int a = 0; a < A_T; ++a)
#pragma unroll
        for (int G = 0; G < 4; ++G)
            if (G < nG) {                            // columns 16 G + 4 c .. + 3 (may reach into the row's padding: ldT >= mp8 + 8)
                *reinterpret_cast<double2*>(tp[a] + 16 * G + 4 * c) = make_double2(acc[a][G][0][0], acc[a][G][1][0]);
                *reinterpret_cast<double2*>(tp[a] + 16 * G + 4 * c + 2) = make_double2(acc[a][G][0][1], acc[a][G][1][1]);
            }
    __syncwarp();
}

// ---------------------------------------------------------------------------
// One tile of one flush job of walker b (the unit of work a CTA takes from the
// walker's ticket word, qmcd_kernel.cuh).  Job phases:
//   0 (K <= 64): row tile, entirely local:  T = -(B C^T - E_J);  T <- T M;  B += T W
//   1 (K >  64): 64-column tile of Y = M W
//   2 (K >  64): row tile with the finished Y:  T = -(B C^T - E_J);  B += T Y
// `mf_key` caches which job's M sits in this CTA's Mf area (phase 0).
// ---------------------------------------------------------------------------
#define QMCD_JOB_LOCAL 0
#define QMCD_JOB_Y 1
#define QMCD_JOB_ROWS_Y 2
#define QMCD_Y_TILE_COLS 64

__host__ __device__ inline int qmcd_job_ntiles(int N, int tile_rows, int phase) {
    return (phase == QMCD_JOB_Y) ? N / QMCD_Y_TILE_COLS : (N + tile_rows - 1) / tile_rows;
}

template <int A_T, int NS>
__device__ void qmcd_flush_tile_impl(const QmcdDev& P, unsigned char* dyn, int b, int phase, int m, int tile,
                                     unsigned long long job_key, unsigned long long& mf_key) {
    constexpr int R = 64 * A_T;
    const int N = P.N, K = P.K, tid = threadIdx.x;
    const int ldT = qmcd_mma_ldT(K);
    const int mp8 = (m + 7) & ~7;
    double* Ts = reinterpret_cast<double*>(dyn);
    double* cb = Ts + (size_t)qmcd_mma_rows(K) * ldT;
    double* Bw = P.B + (size_t)b * N * N;
    const double* Cw = P.C + (size_t)b * K * N;
    const double* Ww = P.W + (size_t)b * K * N;
    double* Yw = P.Y + (size_t)b * K * N;
    const double* Mw = P.M + (size_t)b * P.ldMg * P.ldMg;
    const int* Jw = P.J + (size_t)b * K;
    if (phase == QMCD_JOB_LOCAL) {
        double* Mf = cb + (size_t)NS * QMCD_MMA_CHUNK_DOUBLES;
        if (mf_key != job_key) {                       // M of this job is not staged yet in this CTA
            __syncthreads();
            for (int idx = tid; idx < 64 * 64; idx += QMCD_THREADS) {
                const int a = idx >> 6, bb = idx & 63;
                Mf[a * QMCD_MMA_LDX + bb] = (a < m && bb < m) ? __ldcg(Mw + (size_t)a * P.ldMg + bb) : 0.0;
            }
            mf_key = job_key;
        }
        const int row0 = tile * R, nvalid = min(R, N - row0);
        if (mp8 <= 32) qmcd_mma_nt<A_T, 4, NS>(Bw, N, row0, nvalid, Cw, Jw, m, Ts, ldT, cb);
        else qmcd_mma_nt<A_T, 8, NS>(Bw, N, row0, nvalid, Cw, Jw, m, Ts, ldT, cb);
        qmcd_mma_tm<A_T>(Ts, ldT, mp8, Mf);      // (the NT stage ended with a barrier: Mf and Ts are visible)
        qmcd_mma_nn<A_T, true, NS>(Ts, ldT, mp8, Ww, m, N, Bw, row0, nvalid, 0, N, cb);
        __syncthreads();
        return;
    }
    mf_key = 0;                                        // the other phases overwrite the Mf area's neighbours / Ts
    if (phase == QMCD_JOB_Y) {
        // Y[:, c0 .. c0+64) = M W[:, c0 .. c0+64), M taken R rows at a time as the A operand
        const int c0 = tile * QMCD_Y_TILE_COLS;
        for (int r0 = 0; r0 < m; r0 += R) {
            __syncthreads();
            for (int idx = tid; idx < R * mp8; idx += QMCD_THREADS) {
                const int r = idx / mp8, a = idx - r * mp8;
                Ts[(size_t)r * ldT + a] = (r0 + r < m && a < m) ? __ldcg(Mw + (size_t)(r0 + r) * P.ldMg + a) : 0.0;
            }
            __syncthreads();
            qmcd_mma_nn<A_T, false, NS>(Ts, ldT, mp8, Ww, m, N, Yw, r0, min(R, m - r0), c0, c0 + QMCD_Y_TILE_COLS, cb);
        }
        __syncthreads();
        return;
    }
    const int row0 = tile * R, nvalid = min(R, N - row0);
    if (mp8 <= 32) qmcd_mma_nt<A_T, 4, NS>(Bw, N, row0, nvalid, Cw, Jw, m, Ts, ldT, cb);
    else qmcd_mma_nt<A_T, 8, NS>(Bw, N, row0, nvalid, Cw, Jw, m, Ts, ldT, cb);
    qmcd_mma_nn<A_T, true, NS>(Ts, ldT, mp8, Yw, m, N, Bw, row0, nvalid, 0, N, cb);
    __syncthreads();
}

// tile_rows = 128 needs K <= 64 (T for 128 rows beside the chunk ring); the host guarantees it
__device__ inline void qmcd_flush_tile(const QmcdDev& P, unsigned char* dyn, int b, int phase, int m, int tile,
                                       unsigned long long job_key, unsigned long long& mf_key) {
    if (qmcd_mma_stages(P.K) == 3) {
        if (P.tile_rows == 128) qmcd_flush_tile_impl<2, 3>(P, dyn, b, phase, m, tile, job_key, mf_key);
        else qmcd_flush_tile_impl<1, 3>(P, dyn, b, phase, m, tile, job_key, mf_key);
    } else {
        qmcd_flush_tile_impl<1, 2>(P, dyn, b, phase, m, tile, job_key, mf_key);
    }
}
