// qmcd_phases.cuh -- the phases of the hot path as cluster-cooperative device
// functions: look-ahead ratio (F1), accept/border (F2), flush (F3/F4).
// Citations: lines of /root/reference/PAPER.md.
#pragma once
#include "qmcd_dev.cuh"

struct QmcdWalker {          // per-CTA view of the walker this cluster owns
    int b;                   // walker index
    int r;                   // CTA rank in the cluster
    int klo, khi;            // owned column slice (ratio) == owned row slice (flush)
    double *B, *C, *W, *Y, *M;
    int* J;
};

__device__ inline QmcdWalker qmcd_walker(const QmcdDev& P, int b, int r) {
    QmcdWalker w;
    w.b = b; w.r = r;
    w.klo = qmcd_slice_lo(P.N, P.S, r);
    w.khi = qmcd_slice_lo(P.N, P.S, r + 1);
    w.B = P.B + (size_t)b * P.N * P.N;
    w.C = P.C + (size_t)b * P.K * P.N;
    w.W = P.W + (size_t)b * P.K * P.N;
    w.Y = P.Y + (size_t)b * P.K * P.N;
    w.M = P.M + (size_t)b * P.K * P.K;
    w.J = P.J + (size_t)b * P.K;
    return w;
}

// ---------------------------------------------------------------------------
// F1: look-ahead ratio (Eqs. 1 and 3).
//   d = B0[j,:].v ; p_i = B0[j,:].C[i,:] - delta(j,j_i) ; q_a = W[a,:].v
//   R = d - p^T M q                                   (m = 0: R = d)
// Every CTA streams its column slice: 2m+2 vectors of length N/S, fully
// coalesced; partial sums go to the leader CTA's shared memory through DSMEM.
// The slices of B0[j,:] and v are also written to slot m of W and C -- the slot
// the move will occupy if accepted -- so accept has nothing left to copy.
// Returns R in the leader CTA (all threads); other CTAs return 0.
// Ends with the leader's pf (delta applied), cf = M q valid in ITS smem.
// ---------------------------------------------------------------------------
__device__ double qmcd_ratio_phase(const QmcdDev& P, const QmcdSmem& s, cg::cluster_group& cl,
                                   const QmcdWalker& w, int j, int m, const double* __restrict__ v) {
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int N = P.N, K = P.K, S = P.S;
    const int len = w.khi - w.klo;
    const int PL = 2 * K + 1;
    const double* rowj = w.B + (size_t)j * N + w.klo;
    const double* vv = v + w.klo;
    double* Wm = w.W + (size_t)m * N + w.klo;
    double* Cm = w.C + (size_t)m * N + w.klo;

    double dpart = 0.0;
    for (int k = tid; k < len; k += QMCD_THREADS) {
        double rv = qmcd_ldcg(rowj + k);
        double xv = vv[k];
        s.rs[k] = rv; s.vs[k] = xv;
        Wm[k] = rv; Cm[k] = xv;
        dpart += rv * xv;
    }
    dpart = qmcd_warp_sum(dpart);
    if (lane == 0) s.red[wid] = dpart;
    __syncthreads();

    double* lead_part = (S > 1) ? cl.map_shared_rank(s.part, 0) : s.part;
    double* mine = lead_part + (size_t)w.r * PL;
    if (tid == 0) {
        double d = 0.0;
#pragma unroll
        for (int i = 0; i < QMCD_WARPS; ++i) d += s.red[i];
        mine[2 * K] = d;
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
            p0 += rk * qmcd_ldcg(C0 + k);
            q0 += qmcd_ldcg(W0 + k) * vk;
            p1 += rk * qmcd_ldcg(C1 + k);
            q1 += qmcd_ldcg(W1 + k) * vk;
        }
        p0 = qmcd_warp_sum(p0); q0 = qmcd_warp_sum(q0);
        p1 = qmcd_warp_sum(p1); q1 = qmcd_warp_sum(q1);
        if (lane == 0) {
            mine[i] = p0; mine[K + i] = q0;
            if (two) { mine[i + 1] = p1; mine[K + i + 1] = q1; }
        }
    }
    if (S > 1) cl.sync(); else __syncthreads();
    if (w.r != 0) return 0.0;

    // ---- leader: reduce partials, c = M q, R = d - p.c
    for (int i = tid; i < m; i += QMCD_THREADS) {
        double p = 0, q = 0;
        for (int r = 0; r < S; ++r) { p += s.part[(size_t)r * PL + i]; q += s.part[(size_t)r * PL + K + i]; }
        if (w.J[i] == j) p -= 1.0;
        s.pf[i] = p; s.qf[i] = q;
    }
    if (tid == 0) {
        double d = 0;
        for (int r = 0; r < S; ++r) d += s.part[(size_t)r * PL + 2 * K];
        s.red[8] = d;
    }
    __syncthreads();
    for (int a = wid; a < m; a += QMCD_WARPS) {
        const double* Ma = w.M + (size_t)a * K;
        double acc = 0;
        for (int bb = lane; bb < m; bb += 32) acc += qmcd_ldcg(Ma + bb) * s.qf[bb];
        acc = qmcd_warp_sum(acc);
        if (lane == 0) s.cf[a] = acc;
    }
    __syncthreads();
    if (wid == 0) {
        double acc = 0;
        for (int a = lane; a < m; a += 32) acc += s.pf[a] * s.cf[a];
        acc = qmcd_warp_sum(acc);
        if (lane == 0) s.red[9] = s.red[8] - acc;
    }
    __syncthreads();
    return s.red[9];
}

// ---------------------------------------------------------------------------
// F2: accept = border M.  With S_new = [[S, q],[p^T, d]]
// and Schur complement R = d - p^T M q:
//   M_new = [[M + sigma c r^T, -sigma c], [-sigma r^T, sigma]],
//   c = M q, r^T = p^T M, sigma = 1/R.
// Leader CTA only; pf/cf must be valid in its smem (delta term is zero because
// the caller flushes first when j is already queued).  C[m], W[m] were staged by
// the ratio phase.
// ---------------------------------------------------------------------------
__device__ void qmcd_accept_update(const QmcdDev& P, const QmcdSmem& s, const QmcdWalker& w,
                                   int j, int m, double R) {
    const int tid = threadIdx.x;
    const int K = P.K;
    const double sigma = 1.0 / R;
    for (int bb = tid; bb < m; bb += QMCD_THREADS) {
        double acc = 0;
        for (int a = 0; a < m; ++a) acc += s.pf[a] * qmcd_ldcg(w.M + (size_t)a * K + bb);
        s.rf[bb] = acc;
    }
    __syncthreads();
    for (int idx = tid; idx < m * m; idx += QMCD_THREADS) {
        int a = idx / m, bb = idx - a * m;
        double* p = w.M + (size_t)a * K + bb;
        *p = qmcd_ldcg(p) + sigma * s.cf[a] * s.rf[bb];
    }
    for (int a = tid; a < m; a += QMCD_THREADS) {
        w.M[(size_t)a * K + m] = -sigma * s.cf[a];
        w.M[(size_t)m * K + a] = -sigma * s.rf[a];
    }
    if (tid == 0) {
        w.M[(size_t)m * K + m] = sigma;
        w.J[m] = j;
        P.m[w.b] = m + 1;
        P.sj[w.b] = -1;
        P.counters[(size_t)w.b * 2 + 0] += 1;
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
            const double* Ma = w.M + (size_t)a * K;
            double acc = 0;
            for (int bb = 0; bb < m; ++bb) acc += qmcd_ldcg(Ma + bb) * qmcd_ldcg(w.W + (size_t)bb * N + k);
            w.Y[(size_t)a * N + k] = acc;
        }
    }
    if (S > 1) cl.sync(); else __syncthreads();
    // steps 2-3: rows of my slice, one warp per row
    double* Tw = s.Ts + (size_t)wid * K;
    for (int r = w.klo + wid; r < w.khi; r += QMCD_WARPS) {
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
                if (lane == 0 && u < na) Tw[a0 + u] = t - ((w.J[a0 + u] == r) ? 1.0 : 0.0);
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
