// qmcd_flush_mma.cuh -- FP64 tensor-core (DMMA) flush of Eq. 4:
//     Y = M W            (m x N,  by column slice, one cluster sync after it)
//     T = B0 C^T - E_J   (row tile x m, reduction over N)          "NT stage"
//     B <- B0 - T Y      (row tile x N, reduction over m)          "NN stage"
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
__host__ __device__ inline size_t qmcd_flush_mma_smem_bytes(int N, int K) {
    (void)N;
    return (size_t)qmcd_mma_rows(K) * qmcd_mma_ldT(K) * 8 + 2 * (size_t)QMCD_MMA_CHUNK_DOUBLES * 8;
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

__device__ inline bool qmcd_flush_use_mma(const QmcdDev& P, int m) {
    if (P.flush_path == 1) return false;
    const bool ok = (P.N % 64 == 0) && ((P.N / P.S) % 64 == 0) && P.mma_smem_ok;
    if (!ok) return false;
    if (P.flush_path == 2) return true;
    return m >= 2;
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

__device__ __forceinline__ double2 qmcd_lds128(const double* p) { return *reinterpret_cast<const double2*>(p); }
// coherent (never .nc) 16-byte global load / store of B: the same kernel rewrites B
__device__ __forceinline__ double2 qmcd_ldg128(const double* p) {
    double2 v;
    asm volatile("ld.global.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p) : "memory");
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
template <int A_T, int NB>
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
        qmcd_stage_chunk<QMCD_MMA_LDC>(cb, Cq, (size_t)N, col0, ncols, m, 0);
        qmcd_cp_async_commit();
        double2 a_next[A_T];
#pragma unroll
        for (int a = 0; a < A_T; ++a) a_next[a] = av[a] ? qmcd_ldg128(ap[a]) : make_double2(0.0, 0.0);
        for (int kc = 0; kc < nchunks; ++kc) {
            if (kc + 1 < nchunks) {
                qmcd_stage_chunk<QMCD_MMA_LDC>(cb + ((kc + 1) & 1) * QMCD_MMA_CHUNK_DOUBLES, Cq, (size_t)N, col0, ncols, m,
                                               (kc + 1) * QMCD_MMA_KC);
                qmcd_cp_async_commit();
                qmcd_cp_async_wait<1>();
            } else {
                qmcd_cp_async_wait<0>();
            }
            __syncthreads();
            const double* cur = cb + (kc & 1) * QMCD_MMA_CHUNK_DOUBLES + g * QMCD_MMA_LDC + 2 * c;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                double2 a_cur[A_T];
#pragma unroll
                for (int a = 0; a < A_T; ++a) a_cur[a] = a_next[a];
                const int nk = kc * QMCD_MMA_KC + (q + 1) * 8;
                if (nk < N) {
#pragma unroll
                    for (int a = 0; a < A_T; ++a)
                        if (av[a]) a_next[a] = qmcd_ldg128(ap[a] + nk);
                }
                // all k-step-0 MMAs, then all k-step-1 MMAs: consecutive DMMAs are independent
                double2 bv[NB];
#pragma unroll
                for (int b = 0; b < NB; ++b) bv[b] = qmcd_lds128(cur + b * 8 * QMCD_MMA_LDC + 8 * q);
#pragma unroll
                for (int b = 0; b < NB; ++b)
#pragma unroll
                    for (int a = 0; a < A_T; ++a) qmcd_dmma(acc[a][b][0], acc[a][b][1], a_cur[a].x, bv[b].x);
#pragma unroll
                for (int b = 0; b < NB; ++b)
#pragma unroll
                    for (int a = 0; a < A_T; ++a) qmcd_dmma(acc[a][b][0], acc[a][b][1], a_cur[a].y, bv[b].y);
            }
            __syncthreads();
        }
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
// (cp.async, double buffered over the linear (n-chunk, k-chunk) sequence); the
// warp's 16 A_T/2... rows x 64 columns of D live in registers.
// ---------------------------------------------------------------------------
template <int A_T, bool INIT>
__device__ void qmcd_mma_nn(const double* __restrict__ Ts, int ldT, int kext,
                            const double* __restrict__ X, int m_valid, int N,
                            double* D, int row0, int nvalid, int c_lo, int c_hi,
                            double* __restrict__ cb) {
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, g = lane >> 2, c = lane & 3;
    const int nk = (kext + 63) >> 6;
    const int nn = (c_hi - c_lo) >> 6;
    const int total = nn * nk;
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
    qmcd_stage_chunk<QMCD_MMA_LDX>(cb, X, (size_t)N, 0, min(64, kext), m_valid, c_lo);
    qmcd_cp_async_commit();
    int ci = 0;
    for (int ni = 0; ni < nn; ++ni) {
        const int n0 = c_lo + ni * 64;
        double2 binit[A_T][4][2];
        if (INIT) {
#pragma unroll
            for (int a = 0; a < A_T; ++a)
#pragma unroll
                for (int G = 0; G < 4; ++G) {
                    binit[a][G][0] = rv[a] ? qmcd_ldg128(dp[a] + n0 + 16 * G) : make_double2(0.0, 0.0);
                    binit[a][G][1] = rv[a] ? qmcd_ldg128(dp[a] + n0 + 16 * G + 2) : make_double2(0.0, 0.0);
                }
        }
        double acc[A_T][4][2][2];
#pragma unroll
        for (int a = 0; a < A_T; ++a)
#pragma unroll
            for (int G = 0; G < 4; ++G) { acc[a][G][0][0] = acc[a][G][0][1] = acc[a][G][1][0] = acc[a][G][1][1] = 0.0; }
        for (int kb = 0; kb < nk; ++kb, ++ci) {
            if (ci + 1 < total) {
                const int nci = ci + 1, nni = nci / nk, nkb = nci - nni * nk;
                qmcd_stage_chunk<QMCD_MMA_LDX>(cb + (nci & 1) * QMCD_MMA_CHUNK_DOUBLES, X, (size_t)N, nkb * 64,
                                               min(64, kext - nkb * 64), m_valid, c_lo + nni * 64);
                qmcd_cp_async_commit();
                qmcd_cp_async_wait<1>();
            } else {
                qmcd_cp_async_wait<0>();
            }
            __syncthreads();
            const double* cur = cb + (ci & 1) * QMCD_MMA_CHUNK_DOUBLES + (2 * c) * QMCD_MMA_LDX + 2 * g;
            const int nq = min(64, kext - kb * 64) >> 3;
#pragma unroll 2
            for (int q = 0; q < nq; ++q) {
                double2 avv[A_T];
#pragma unroll
                for (int a = 0; a < A_T; ++a) avv[a] = qmcd_lds128(tp[a] + kb * 64 + 8 * q);
                double2 x0[4], x1[4];
#pragma unroll
                for (int G = 0; G < 4; ++G) {
                    x0[G] = qmcd_lds128(cur + (8 * q) * QMCD_MMA_LDX + 16 * G);
                    x1[G] = qmcd_lds128(cur + (8 * q + 1) * QMCD_MMA_LDX + 16 * G);
                }
#pragma unroll
                for (int G = 0; G < 4; ++G)
#pragma unroll
                    for (int a = 0; a < A_T; ++a) {
                        qmcd_dmma(acc[a][G][0][0], acc[a][G][0][1], avv[a].x, x0[G].x);
                        qmcd_dmma(acc[a][G][1][0], acc[a][G][1][1], avv[a].x, x0[G].y);
                    }
#pragma unroll
                for (int G = 0; G < 4; ++G)
#pragma unroll
                    for (int a = 0; a < A_T; ++a) {
                        qmcd_dmma(acc[a][G][0][0], acc[a][G][0][1], avv[a].y, x1[G].x);
                        qmcd_dmma(acc[a][G][1][0], acc[a][G][1][1], avv[a].y, x1[G].y);
                    }
            }
            __syncthreads();
        }
#pragma unroll
        for (int a = 0; a < A_T; ++a) {
            if (!rv[a]) continue;
#pragma unroll
            for (int G = 0; G < 4; ++G) {
                double o0 = acc[a][G][0][0], o1 = acc[a][G][1][0], o2 = acc[a][G][0][1], o3 = acc[a][G][1][1];
                if (INIT) { o0 += binit[a][G][0].x; o1 += binit[a][G][0].y; o2 += binit[a][G][1].x; o3 += binit[a][G][1].y; }
                qmcd_stg128(dp[a] + n0 + 16 * G, o0, o1);
                qmcd_stg128(dp[a] + n0 + 16 * G + 2, o2, o3);
            }
        }
    }
}

template <int A_T>
__device__ void qmcd_flush_mma_impl(const QmcdDev& P, const QmcdSmem& s, cg::cluster_group& cl,
                                    const QmcdWalker& w, int m) {
    constexpr int R = 64 * A_T;
    const int N = P.N, K = P.K, tid = threadIdx.x;
    const int ldT = qmcd_mma_ldT(K);
    const int mp8 = (m + 7) & ~7;
    double* Ts = reinterpret_cast<double*>(s.dyn);
    double* cb = Ts + (size_t)qmcd_mma_rows(K) * ldT;
    // ---- Y = M W on my column slice, M taken R rows at a time as the A operand
    for (int r0 = 0; r0 < m; r0 += R) {
        for (int idx = tid; idx < R * mp8; idx += QMCD_THREADS) {
            const int r = idx / mp8, a = idx - r * mp8;
            Ts[(size_t)r * ldT + a] = (r0 + r < m && a < m) ? __ldcg(w.M + (size_t)(r0 + r) * K + a) : 0.0;
        }
        __syncthreads();
        qmcd_mma_nn<A_T, false>(Ts, ldT, mp8, w.W, m, N, w.Y, r0, min(R, m - r0), w.klo, w.khi, cb);
        __syncthreads();
    }
    if (P.S > 1) cl.sync(); else __syncthreads();
    // ---- my row slice, R rows at a time:  T = -(B C^T - E_J);  B += T Y
    for (int row0 = w.klo; row0 < w.khi; row0 += R) {
        const int nvalid = min(R, w.khi - row0);
        if (mp8 <= 32) qmcd_mma_nt<A_T, 4>(w.B, N, row0, nvalid, w.C, w.J, m, Ts, ldT, cb);
        else qmcd_mma_nt<A_T, 8>(w.B, N, row0, nvalid, w.C, w.J, m, Ts, ldT, cb);
        qmcd_mma_nn<A_T, true>(Ts, ldT, mp8, w.Y, m, N, w.B, row0, nvalid, 0, N, cb);
        __syncthreads();
    }
}

__device__ inline void qmcd_flush_mma(const QmcdDev& P, const QmcdSmem& s, cg::cluster_group& cl,
                                      const QmcdWalker& w, int m) {
    if (qmcd_mma_rows(P.K) == 128 && (w.khi - w.klo) >= 128) qmcd_flush_mma_impl<2>(P, s, cl, w, m);
    else qmcd_flush_mma_impl<1>(P, s, cl, w, m);
}
