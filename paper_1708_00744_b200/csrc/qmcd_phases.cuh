// qmcd_phases.cuh -- the phases of the hot path as cluster-cooperative device
// functions: look-ahead ratio (F1), accept/border (F2), flush (F3/F4).
// Citations: lines of /root/reference/PAPER.md.
#pragma once
#include "qmcd_dev.cuh"

struct QmcdWalker {          // per-CTA view of the walker this (leader) cluster works for
    int b;                   // walker index
    int r;                   // CTA rank in the cluster
    int klo, khi;            // column slice of the look-ahead and of the CUDA-core flush's Y = M W
    int rlo, rhi;            // row slice of B in the CUDA-core flush (over the S CTAs of the cluster)
    double *B, *C, *W, *Y, *M;
    int* J;
};

__device__ inline QmcdWalker qmcd_walker(const QmcdDev& P, int b, int r) {
    QmcdWalker w;
    w.b = b; w.r = r;
    w.klo = qmcd_slice_lo(P.N, P.S, r);
    w.khi = qmcd_slice_lo(P.N, P.S, r + 1);
    w.rlo = w.klo; w.rhi = w.khi;
    w.B = P.B + (size_t)b * P.N * P.N;
    w.C = P.C + (size_t)b * P.K * P.N;
    w.W = P.W + (size_t)b * P.K * P.N;
    w.Y = P.Y + (size_t)b * P.K * P.N;
    w.M = P.M + (size_t)b * P.ldMg * P.ldMg;
    w.J = P.J + (size_t)b * P.K;
    return w;
}

// M lives either in every CTA's shared memory (MS = true: s.Ms, row stride K|1,
// identical copies kept in step by identical arithmetic) or, when K is too large
// for that, in global memory (w.M, row stride P.ldMg, written by the leader CTA only).
template <bool MS> struct QmcdM {
    static __device__ __forceinline__ const double* base(const QmcdSmem& s, const QmcdWalker& w) { return MS ? s.Ms : w.M; }
    static __device__ __forceinline__ int ld(const QmcdDev& P) { return MS ? qmcd_ldM(P.K) : P.ldMg; }
    static __device__ __forceinline__ double get(const double* p) { return MS ? *p : __ldcg(p); }
};

__device__ __forceinline__ void qmcd_prefetch_l2(const void* p) {
    asm volatile("prefetch.global.L2 [%0];" :: "l"(p));
}

// ---------------------------------------------------------------------------
// F1: look-ahead ratio (Eqs. 1 and 3).
//   d = B0[j,:].v ; p_i = B0[j,:].C[i,:] - delta(j,j_i) ; q_a = W[a,:].v
//   R = d - p^T M q                                   (m = 0: R = d)
// Every CTA streams its column slice (2m+2 vectors of length N/S, coalesced) and
// sends its partial sums to EVERY CTA of the cluster through distributed shared
// memory; after ONE cluster barrier each CTA reduces them in the same order and
// finishes the K x K part on its own, so all CTAs hold bit-identical R, c = M q
// and r = M^T p and take the accept decision without another exchange.
// The slices of B0[j,:] and v are also written to slot m of W and C -- the slot
// the move will occupy if accepted.  `pbuf` is the partial-buffer parity, toggled
// here.  Returns R in every thread; *inq = (j is already queued).
// ---------------------------------------------------------------------------
template <bool MS>
__device__ double qmcd_lookahead(const QmcdDev& P, const QmcdSmem& s, cg::cluster_group& cl,
                                 const QmcdWalker& w, int j, int m, const double* v,
                                 int& pbuf, bool* inq) {
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int N = P.N, K = P.K, S = P.S;
    const int len = w.khi - w.klo;
    const int PL = qmcd_PL(K);
    const double* rowj = w.B + (size_t)j * N + w.klo;
    const double* vv = v + w.klo;
    double* Wm = w.W + (size_t)m * N + w.klo;
    double* Cm = w.C + (size_t)m * N + w.klo;
    const int buf = pbuf;
    pbuf ^= 1;

    double dpart = 0.0;
    for (int k = tid; k < len; k += QMCD_THREADS) {
        double rv = __ldcg(rowj + k);
        double xv = __ldcg(vv + k);
        s.rs[k] = rv; s.vs[k] = xv;
        Wm[k] = rv; Cm[k] = xv;
        dpart += rv * xv;
    }
    dpart = qmcd_warp_sum(dpart);
    if (lane == 0) s.red[wid] = dpart;
    __syncthreads();

    // my partials go to slot [buf][w.r] of every CTA q (lane q of each warp stores)
    double* dst = nullptr;
    if (lane < S) dst = ((S > 1) ? cl.map_shared_rank(s.part, lane) : s.part) + ((size_t)buf * S + w.r) * PL;
    if (wid == 0) {
        double d = 0.0;
#pragma unroll
        for (int i = 0; i < QMCD_WARPS; ++i) d += s.red[i];
        if (lane < S) dst[2 * K] = d;
    }
    // dots: each warp takes two queue rows at a time (4 independent streams)
    for (int i = wid * 2; i < m; i += QMCD_WARPS * 2) {
        const bool two = (i + 1 < m);
        const double* C0 = w.C + (size_t)i * N + w.klo;
        const double* W0 = w.W + (size_t)i * N + w.klo;
        const double* C1 = two ? C0 + N : C0;
        const double* W1 = two ? W0 + N : W0;
        double p0 = 0, q0 = 0, p1 = 0, q1 = 0;
#pragma unroll 4
        for (int k = lane; k < len; k += 32) {
            double rk = s.rs[k], vk = s.vs[k];
            p0 += rk * __ldcg(C0 + k);
            q0 += __ldcg(W0 + k) * vk;
            p1 += rk * __ldcg(C1 + k);
            q1 += __ldcg(W1 + k) * vk;
        }
        p0 = qmcd_warp_sum(p0); q0 = qmcd_warp_sum(q0);
        p1 = qmcd_warp_sum(p1); q1 = qmcd_warp_sum(q1);
        if (lane < S) {
            dst[i] = p0; dst[K + i] = q0;
            if (two) { dst[i + 1] = p1; dst[K + i + 1] = q1; }
        }
    }
    if (S > 1) cl.sync(); else __syncthreads();

    // ---- every CTA: reduce the S partial vectors in rank order
    const double* mypart = s.part + (size_t)buf * S * PL;
    for (int i = tid; i < m; i += QMCD_THREADS) {
        double p = 0, q = 0;
        for (int r = 0; r < S; ++r) { p += mypart[(size_t)r * PL + i]; q += mypart[(size_t)r * PL + K + i]; }
        if (s.Js[i] == j) p -= 1.0;
        s.pf[i] = p; s.qf[i] = q;
    }
    double d = 0;
    for (int r = 0; r < S; ++r) d += mypart[(size_t)r * PL + 2 * K];
    __syncthreads();
    // ---- c = M q and r = M^T p: 8 threads per index x, strided partial sums
    {
        const double* Mb = QmcdM<MS>::base(s, w);
        const int ldM = QmcdM<MS>::ld(P);
        const int h = tid & 7;
        for (int x0 = 0; x0 < m; x0 += QMCD_THREADS / 8) {
            const int x = x0 + (tid >> 3);
            double ca = 0, ra = 0;
            if (x < m) {
                for (int b = h; b < m; b += 8) {
                    ca += QmcdM<MS>::get(Mb + (size_t)x * ldM + b) * s.qf[b];
                    ra += s.pf[b] * QmcdM<MS>::get(Mb + (size_t)b * ldM + x);
                }
            }
#pragma unroll
            for (int o = 4; o > 0; o >>= 1) {
                ca += __shfl_xor_sync(0xffffffffu, ca, o);
                ra += __shfl_xor_sync(0xffffffffu, ra, o);
            }
            if (x < m && h == 0) { s.cf[x] = ca; s.rf[x] = ra; }
        }
    }
    __syncthreads();
    // ---- every warp: R = d - p.c, and whether j is already queued
    double acc = 0;
    bool q_in = false;
    for (int a = lane; a < m; a += 32) { acc += s.pf[a] * s.cf[a]; q_in |= (s.Js[a] == j); }
    acc = qmcd_warp_sum(acc);
    if (inq) *inq = __any_sync(0xffffffffu, q_in);
    return d - acc;
}

// ---------------------------------------------------------------------------
// F2: accept = border M.  With S_new = [[S, q],[p^T, d]]
// and Schur complement R = d - p^T M q:
//   M_new = [[M + sigma c r^T, -sigma c], [-sigma r^T, sigma]],
//   c = M q, r^T = p^T M, sigma = 1/R.
// cf / rf must be valid in shared memory (the delta term is zero because the
// caller flushes first when j is already queued).  C[m], W[m] were staged by the
// look-ahead.  MS: every CTA updates its own copy; otherwise the leader only.
// ---------------------------------------------------------------------------
template <bool MS>
__device__ void qmcd_accept_update(const QmcdDev& P, const QmcdSmem& s, const QmcdWalker& w,
                                   int j, int m, double R) {
    const int tid = threadIdx.x;
    const double sigma = 1.0 / R;
    if (MS || w.r == 0) {
        double* Mb = MS ? s.Ms : w.M;
        const int ldM = QmcdM<MS>::ld(P);
        for (int idx = tid; idx < m * m; idx += QMCD_THREADS) {
            int a = idx / m, bb = idx - a * m;
            double* p = Mb + (size_t)a * ldM + bb;
            *p = QmcdM<MS>::get(p) + sigma * s.cf[a] * s.rf[bb];
        }
        for (int a = tid; a < m; a += QMCD_THREADS) {
            Mb[(size_t)a * ldM + m] = -sigma * s.cf[a];
            Mb[(size_t)m * ldM + a] = -sigma * s.rf[a];
        }
        if (tid == 0) Mb[(size_t)m * ldM + m] = sigma;
    }
    if (tid == 0) {
        s.Js[m] = j;
        if (w.r == 0) {
            w.J[m] = j;
            P.counters[(size_t)w.b * 8 + 0] += 1;
        }
    }
    __syncthreads();
}

// ---------------------------------------------------------------------------
// F2, repeated electron (reading G7, second alternative; the paper is silent):
// electron j = J[a] is accepted again before the queue was applied.  The current matrix is A0 with
// column j = the NEWEST column, so slot a keeps its row W[a,:] = B0[j,:] and only its column changes,
// C[a,:] <- v.  S = W C^T changes in column a (to q = W v), and by Sherman-Morrison on that column
//     M' = M - (c - e_a) M[a,:] / c_a,      c = M q,   c_a = M[a,:] q = R  (the ratio of this move).
// cf = c must be valid in shared memory; v sits in slot m of C (staged by the look-ahead).  m, J, W
// are unchanged.  s.rf is used as scratch for the old row a.  Every CTA copies its column slice.
// ---------------------------------------------------------------------------
template <bool MS>
__device__ void qmcd_accept_replace(const QmcdDev& P, const QmcdSmem& s, const QmcdWalker& w,
                                    int a, int m, double R) {
    const int tid = threadIdx.x;
    const double inv = 1.0 / R;
    if (MS || w.r == 0) {
        double* Mb = MS ? s.Ms : w.M;
        const int ldM = QmcdM<MS>::ld(P);
        for (int y = tid; y < m; y += QMCD_THREADS) s.rf[y] = QmcdM<MS>::get(Mb + (size_t)a * ldM + y);
        __syncthreads();
        for (int idx = tid; idx < m * m; idx += QMCD_THREADS) {
            const int x = idx / m, y = idx - x * m;
            double* p = Mb + (size_t)x * ldM + y;
            *p = QmcdM<MS>::get(p) - (s.cf[x] - (x == a ? 1.0 : 0.0)) * s.rf[y] * inv;
        }
    }
    const double* src = w.C + (size_t)m * P.N;
    double* dst = w.C + (size_t)a * P.N;
    for (int k = w.klo + tid; k < w.khi; k += QMCD_THREADS) dst[k] = __ldcg(src + k);
    if (tid == 0 && w.r == 0) P.counters[(size_t)w.b * 8 + 0] += 1;
    __syncthreads();
}

// Leader: copy this walker's M from shared to global memory (before a flush, or
// at the end of a launch).  No-op when M already lives in global memory.
template <bool MS>
__device__ void qmcd_writeback_M(const QmcdDev& P, const QmcdSmem& s, const QmcdWalker& w, int m) {
    if (!MS || w.r != 0) return;
    const int K = P.K, ldM = qmcd_ldM(K);
    for (int idx = threadIdx.x; idx < m * m; idx += QMCD_THREADS) {
        int a = idx / m, bb = idx - a * m;
        w.M[(size_t)a * P.ldMg + bb] = s.Ms[(size_t)a * ldM + bb];
    }
}

// Leader CTA, before a TMA-fed flush (P.use_tma): the 64 x 64 tile of M in global memory must be zero
// outside its valid m x m block (the flush multiplies by the whole zero-padded tile; entries of an
// earlier, longer window may still sit there).
__device__ void qmcd_zero_pad_M(const QmcdDev& P, const QmcdWalker& w, int m) {
    if (w.r != 0) return;
    for (int idx = threadIdx.x; idx < 64 * 64; idx += QMCD_THREADS) {
        const int a = idx >> 6, bb = idx & 63;
        if (a >= m || bb >= m) w.M[(size_t)a * 64 + bb] = 0.0;
    }
}

// Every CTA: load the walker's queue state (J and, if MS, M) into shared memory.
template <bool MS>
__device__ void qmcd_load_state(const QmcdDev& P, const QmcdSmem& s, const QmcdWalker& w, int m) {
    const int K = P.K, ldM = qmcd_ldM(K);
    for (int i = threadIdx.x; i < m; i += QMCD_THREADS) s.Js[i] = __ldcg(w.J + i);
    if (MS)
        for (int idx = threadIdx.x; idx < m * m; idx += QMCD_THREADS) {
            int a = idx / m, bb = idx - a * m;
            s.Ms[(size_t)a * ldM + bb] = __ldcg(w.M + (size_t)a * P.ldMg + bb);
        }
    __syncthreads();
}

// ---------------------------------------------------------------------------
// F3 (CUDA-core path; also the K=1 Sherman-Morrison path F4): Eq. 4,
// PAPER.md:84-89.   Y = M W ; T = B0 C^T - E_J ; B <- B0 - T Y.
// Step 1 by column slice, steps 2-3 by row slice (row-local: one warp per row).
// ---------------------------------------------------------------------------
__device__ void qmcd_flush_simt(const QmcdDev& P, const QmcdSmem& s, cg::cluster_group& cl,
                                const QmcdWalker& w, int m) {
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int N = P.N, K = P.K, S = P.S;
    // step 1: Y[a][k] = sum_b M[a][b] W[b][k], k in my column slice
    for (int k = w.klo + tid; k < w.khi; k += QMCD_THREADS) {
        for (int a = 0; a < m; ++a) {
            const double* Ma = w.M + (size_t)a * P.ldMg;
            double acc = 0;
            for (int bb = 0; bb < m; ++bb) acc += qmcd_ldcg(Ma + bb) * qmcd_ldcg(w.W + (size_t)bb * N + k);
            w.Y[(size_t)a * N + k] = acc;
        }
    }
    if (S > 1) cl.sync(); else __syncthreads();
    // steps 2-3: rows of my slice, one warp per row
    double* Tw = s.Ts + (size_t)wid * K;
    for (int r = w.rlo + wid; r < w.rhi; r += QMCD_WARPS) {
        double* Br = w.B + (size_t)r * N;
        for (int a0 = 0; a0 < m; a0 += 4) {
            double acc[4] = {0, 0, 0, 0};
            const int na = min(4, m - a0);
            for (int k = lane; k < N; k += 32) {
                double bv = qmcd_ldcg(Br + k);
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (u < na) acc[u] += bv * qmcd_ldcg(w.C + (size_t)(a0 + u) * N + k);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                double t = qmcd_warp_sum(acc[u]);
                if (lane == 0 && u < na) Tw[a0 + u] = t - ((__ldcg(w.J + a0 + u) == r) ? 1.0 : 0.0);
            }
        }
        __syncwarp();
        for (int k = lane; k < N; k += 32) {
            double acc = 0;
            for (int a = 0; a < m; ++a) acc += Tw[a] * qmcd_ldcg(w.Y + (size_t)a * N + k);
            Br[k] = qmcd_ldcg(Br + k) - acc;
        }
        __syncwarp();
    }
}
