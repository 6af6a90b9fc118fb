// qmcd_kernel.cuh -- the one __global__ entry: a cluster per walker runs either
// one phase (per-call API) or the whole move loop (qmcd_sweep, persistent).
#pragma once
#include "qmcd_phases.cuh"
#include "qmcd_flush_mma.cuh"

// Flush wrapper: all CTAs of the cluster call it with the same m > 0.
// Barriers: (entry) queue slots / M written by other CTAs become visible;
// (exit) nobody restages slot 0 or reads B rows before every CTA is done.
__device__ void qmcd_flush_phase(const QmcdDev& P, const QmcdSmem& s, cg::cluster_group& cl,
                                 const QmcdWalker& w, int m) {
    if (P.S > 1) cl.sync(); else __syncthreads();
    if (qmcd_flush_use_mma(P, m)) qmcd_flush_mma(P, s, cl, w, m);
    else qmcd_flush_simt(P, s, cl, w, m);
    if (w.r == 0 && threadIdx.x == 0) {
        P.m[w.b] = 0;
        P.counters[(size_t)w.b * 2 + 1] += 1;
    }
    if (P.S > 1) cl.sync(); else __syncthreads();
}

// Is electron j already queued?  (uniform over the cluster: J, m are stable here)
__device__ inline bool qmcd_in_queue(const QmcdWalker& w, int j, int m) {
    for (int i = 0; i < m; ++i)
        if (__ldcg(w.J + i) == j) return true;
    return false;
}

// Accept path shared by ACCEPT and SWEEP.  Called by ALL CTAs with the same
// (j, m, R); pf/cf valid in the leader.  Returns the new m.
__device__ int qmcd_do_accept(const QmcdDev& P, const QmcdSmem& s, cg::cluster_group& cl,
                              const QmcdWalker& w, int j, int m, double R, bool leader_has_R) {
    if (m > 0 && qmcd_in_queue(w, j, m)) {
        // repeated electron inside one window (G7): flush, then the move
        // is re-evaluated against the fresh inverse (m = 0) and queued.  Its v sits
        // in slot m of C (staged by the ratio phase); slot 0 is free after the flush.
        qmcd_flush_phase(P, s, cl, w, m);
        double R2 = qmcd_ratio_phase(P, s, cl, w, j, 0, w.C + (size_t)m * P.N);
        if (w.r == 0) R = R2;
        m = 0;
    }
    if (w.r == 0) qmcd_accept_update(P, s, w, j, m, R);
    m += 1;
    if (m == P.K) { qmcd_flush_phase(P, s, cl, w, m); m = 0; }
    return m;
}

__global__ void __launch_bounds__(QMCD_THREADS, 1) qmcd_kernel(const QmcdArgs A) {
    extern __shared__ __align__(1024) unsigned char qmcd_smem_raw[];
    const QmcdDev& P = A.P;
    cg::cluster_group cl = cg::this_cluster();
    const int S = P.S;
    const int r = (S > 1) ? (int)cl.block_rank() : 0;
    const int b = blockIdx.x / S;
    const QmcdSmem s = qmcd_carve(qmcd_smem_raw, P.N, P.K, S);
    const QmcdWalker w = qmcd_walker(P, b, r);
    const int tid = threadIdx.x;
    int m = __ldcg(P.m + b);

    if (A.mode == QMCD_MODE_RATIO) {
        int j = A.jv ? A.jv[b] : A.j;
        if (j < 0 || j >= P.N) {
            if (r == 0 && tid == 0) { qmcd_set_status(P, QMCD_DEV_EINVAL, b, P.counters[(size_t)b * 2]); P.sj[b] = -1; A.R_out[b] = 0.0; }
            return;   // uniform over the cluster
        }
        double R = qmcd_ratio_phase(P, s, cl, w, j, m, A.v + (size_t)b * P.N);
        if (r == 0) {
            for (int i = tid; i < m; i += QMCD_THREADS) { P.sp[(size_t)b * P.K + i] = s.pf[i]; P.sc[(size_t)b * P.K + i] = s.cf[i]; }
            if (tid == 0) { P.sR[b] = R; P.sj[b] = j; A.R_out[b] = R; }
        }
        return;
    }

    if (A.mode == QMCD_MODE_ACCEPT) {
        const int j = __ldcg(P.sj + b);
        if (j < 0) return;
        const double R = __ldcg(P.sR + b);
        bool acc;
        if (A.uniforms) { double pa = fmin(1.0, R * R); acc = A.uniforms[b] < pa; }
        else acc = A.accept_all || (A.mask[b] != 0);
        if (acc && (R == 0.0 || !isfinite(R))) {
            if (r == 0 && tid == 0) qmcd_set_status(P, QMCD_DEV_ESINGULAR, b, P.counters[(size_t)b * 2]);
            acc = false;
        }
        if (r == 0 && tid == 0 && A.acc_out) A.acc_out[b] = acc ? 1 : 0;
        if (!acc) { if (r == 0 && tid == 0) P.sj[b] = -1; return; }
        if (r == 0) {
            for (int i = tid; i < m; i += QMCD_THREADS) { s.pf[i] = P.sp[(size_t)b * P.K + i]; s.cf[i] = P.sc[(size_t)b * P.K + i]; }
            __syncthreads();
        }
        qmcd_do_accept(P, s, cl, w, j, m, R, true);
        return;
    }

    if (A.mode == QMCD_MODE_FLUSH) {
        if (m > 0) qmcd_flush_phase(P, s, cl, w, m);
        return;
    }

    // ---- QMCD_MODE_SWEEP: the whole move loop, no host round trip.
    int* flag = s.iflag;                         // leader's decision, broadcast via DSMEM
    for (int t = 0; t < A.n_moves; ++t) {
        const int j = (A.j_begin + t) % P.N;
        const size_t tb = (size_t)t * P.batch + b;
        double R = qmcd_ratio_phase(P, s, cl, w, j, m, A.v + tb * P.N);
        if (r == 0 && tid == 0) {
            bool acc;
            if (A.uniforms) { double pa = fmin(1.0, R * R); acc = A.uniforms[tb] < pa; }
            else acc = A.mask[tb] != 0;
            if (acc && (R == 0.0 || !isfinite(R))) {
                qmcd_set_status(P, QMCD_DEV_ESINGULAR, b, t);
                acc = false;
            }
            if (A.R_out) A.R_out[tb] = R;
            if (A.acc_out) A.acc_out[tb] = acc ? 1 : 0;
            for (int q = 0; q < S; ++q) {
                int* f = (S > 1) ? cl.map_shared_rank(flag, q) : flag;
                f[0] = acc ? 1 : 0;
            }
        }
        if (S > 1) cl.sync(); else __syncthreads();
        const bool acc = flag[0] != 0;
        if (acc) m = qmcd_do_accept(P, s, cl, w, j, m, R, true);
    }
    if (r == 0 && tid == 0) P.sj[b] = -1;
}
