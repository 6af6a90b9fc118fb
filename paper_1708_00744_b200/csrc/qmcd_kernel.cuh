// qmcd_kernel.cuh -- the two __global__ entries over one body: clusters of S CTAs, G clusters
// per walker.  qmcd_kernel runs one phase (per-call API) or the per-move sweep, qmcd_kernel_sweep
// the blocked sweep (persistent: the whole move loop); helper clusters serve the flushes.
#pragma once
#include "qmcd_phases.cuh"
#include "qmcd_flush_mma.cuh"

// Eq. 4 on this CTA's row slice (either path); ends with every CTA of the CLUSTER done.
__device__ void qmcd_flush_rows(const QmcdDev& P, const QmcdSmem& s, cg::cluster_group& cl,
                                const QmcdWalker& w, int m) {
    if (qmcd_flush_use_mma(P, m, P.G_act)) qmcd_flush_mma(P, s, cl, w, m);
    else qmcd_flush_simt(P, s, cl, w, m);
}

// Flush wrapper for the LEADER cluster: all its CTAs call it with the same m > 0.
// M goes back to global memory first (the flush reads it from there).  With
// G_act > 1 the walker's helper clusters are released through the `go` word
// (they own the other row slices) and awaited through their `done` words.
// Barriers: (entry) queue slots / M written by other CTAs become visible;
// (exit) nobody restages slot 0 or reads B rows before every CTA is done.
// s.iflag[8] counts the flushes of this launch (same value in every CTA).
template <bool MS>
__device__ void qmcd_flush_phase(const QmcdDev& P, const QmcdSmem& s, cg::cluster_group& cl,
                                 const QmcdWalker& w, int m, bool writeback = true) {
    if (writeback) qmcd_writeback_M<MS>(P, s, w, m);
    if (P.S > 1) cl.sync(); else __syncthreads();
    const int k = s.iflag[8] + 1;
    if (P.G_act > 1 && w.r == 0 && threadIdx.x == 0) {
        __threadfence();
        qmcd_st_release(P.go + w.b, ((unsigned long long)P.launch_id << 32) | ((unsigned long long)k << 12) | (unsigned)m);
    }
    qmcd_flush_rows(P, s, cl, w, m);
    __syncthreads();
    if (threadIdx.x == 0) s.iflag[8] = k;
    if (w.r == 0 && threadIdx.x == 0) {
        P.m[w.b] = 0;
        P.counters[(size_t)w.b * 8 + 1] += 1;
        P.counters[(size_t)w.b * 8 + 7] = 0;          // a new window starts (lock-step proposal count)
        const unsigned long long want = ((unsigned long long)P.launch_id << 32) | (unsigned)k;
        for (int g = 1; g < P.G_act; ++g)
            while (qmcd_ld_acquire(P.done + (size_t)w.b * 16 + g) != want) __nanosleep(20);
    }
    if (P.S > 1) cl.sync(); else __syncthreads();
}

// Helper cluster (w.g > 0): flush my row slices whenever the leader says so, until it says exit.
__device__ void qmcd_helper_loop(const QmcdDev& P, const QmcdSmem& s, cg::cluster_group& cl,
                                 const QmcdWalker& w) {
    for (int k = 1;; ++k) {
        if (threadIdx.x == 0) {
            unsigned long long v;
            for (;;) {
                v = qmcd_ld_acquire(P.go + w.b);
                if ((unsigned)(v >> 32) == P.launch_id) {
                    const unsigned f = (unsigned)(v >> 12) & 0xFFFFFu;
                    if (f == QMCD_GO_EXIT || f == (unsigned)k) break;
                }
                __nanosleep(20);
            }
            s.iflag[9] = (((unsigned)(v >> 12) & 0xFFFFFu) == QMCD_GO_EXIT) ? -1 : (int)(v & 0xFFFu);
        }
        __syncthreads();
        const int m = s.iflag[9];
        if (m < 0) return;
        qmcd_flush_rows(P, s, cl, w, m);
        if (P.S > 1) cl.sync(); else __syncthreads();      // the whole cluster is done with its rows
        if (w.r == 0 && threadIdx.x == 0) {
            __threadfence();
            qmcd_st_release(P.done + (size_t)w.b * 16 + w.g, ((unsigned long long)P.launch_id << 32) | (unsigned)k);
        }
    }
}

#include "qmcd_block.cuh"

// Accept path shared by ACCEPT and SWEEP.  Called by ALL CTAs with the same
// (j, m, R, inq) and cf / rf valid in every CTA.  Returns the new m.
template <bool MS>
__device__ int qmcd_do_accept(const QmcdDev& P, const QmcdSmem& s, cg::cluster_group& cl,
                              const QmcdWalker& w, int j, int m, double R, bool inq, int& pbuf) {
    if (inq) {
        // repeated electron inside one window (G7): flush, then the move
        // is re-evaluated against the fresh inverse (m = 0) and queued.  Its v sits
        // in slot m of C (staged by the look-ahead); slot 0 is free after the flush.
        qmcd_flush_phase<MS>(P, s, cl, w, m);
        R = qmcd_lookahead<MS>(P, s, cl, w, j, 0, w.C + (size_t)m * P.N, pbuf, nullptr);
        m = 0;
    }
    if (!MS && P.S > 1) cl.sync();     // global M: nobody may still be reading it
    qmcd_accept_update<MS>(P, s, w, j, m, R);
    m += 1;
    if (m == P.K) { qmcd_flush_phase<MS>(P, s, cl, w, m); m = 0; }
    return m;
}

template <bool MS>
__device__ void qmcd_run(const QmcdArgs& A, const QmcdSmem& s, cg::cluster_group& cl,
                         const QmcdWalker& w) {
    const QmcdDev& P = A.P;
    const int S = P.S, r = w.r, b = w.b, tid = threadIdx.x;
    int m = __ldcg(P.m + b);   // written by the leader only at the end of a launch or inside a flush
    int pbuf = 0;

    if (A.mode == QMCD_MODE_RATIO) {
        int j = A.jv ? A.jv[b] : A.j;
        if (j < 0 || j >= P.N) {
            if (r == 0 && tid == 0) { qmcd_set_status(P, QMCD_DEV_EINVAL, b, P.counters[(size_t)b * 8]); P.sj[b] = -1; A.R_out[b] = 0.0; }
            return;   // uniform over the cluster
        }
        qmcd_load_state<MS>(P, s, w, m);
        double R = qmcd_lookahead<MS>(P, s, cl, w, j, m, A.v + (size_t)b * P.N, pbuf, nullptr);
        if (r == 0) {
            for (int i = tid; i < m; i += QMCD_THREADS) { P.sc[(size_t)b * P.K + i] = s.cf[i]; P.sr[(size_t)b * P.K + i] = s.rf[i]; }
            if (tid == 0) { P.sR[b] = R; P.sj[b] = j; A.R_out[b] = R; }
        }
        return;
    }

    if (A.mode == QMCD_MODE_ACCEPT) {
        const int j = __ldcg(P.sj + b);
        if (j < 0) return;
        const double R = __ldcg(P.sR + b);
        // lock-step: this proposal takes a slot of the window whatever the decision
        int pw = QMCD_LOCKSTEP(P) ? (int)__ldcg(P.counters + (size_t)b * 8 + 7) + 1 : 0;
        // every CTA has read the staged proposal before the leader clears it
        if (S > 1) cl.sync();
        bool acc;
        if (A.reject_all) acc = false;
        else if (A.uniforms) { double pa = fmin(1.0, R * R); acc = A.uniforms[b] < pa; }
        else acc = A.accept_all || (A.mask[b] != 0);
        if (acc && (R == 0.0 || !isfinite(R))) {
            if (r == 0 && tid == 0) qmcd_set_status(P, QMCD_DEV_ESINGULAR, b, P.counters[(size_t)b * 8]);
            acc = false;
        }
        if (r == 0 && tid == 0) {
            if (A.acc_out) A.acc_out[b] = acc ? 1 : 0;
            P.sj[b] = -1;
        }
        if (!acc) {
            if (QMCD_LOCKSTEP(P)) {
                if (pw >= P.K) {                       // the window is full: Eq. 4 for whatever was accepted in it
                    if (m > 0) qmcd_flush_phase<false>(P, s, cl, w, m);   // M is in global memory between launches
                    pw = 0;
                }
                if (r == 0 && tid == 0) P.counters[(size_t)b * 8 + 7] = pw;
            }
            return;
        }
        qmcd_load_state<MS>(P, s, w, m);
        bool inq = false;
        for (int i = tid; i < m; i += QMCD_THREADS) {
            s.cf[i] = __ldcg(P.sc + (size_t)b * P.K + i); s.rf[i] = __ldcg(P.sr + (size_t)b * P.K + i);
        }
        for (int i = 0; i < m; ++i) inq |= (s.Js[i] == j);
        __syncthreads();
        m = qmcd_do_accept<MS>(P, s, cl, w, j, m, R, inq, pbuf);
        if (QMCD_LOCKSTEP(P)) {
            if (inq) pw = 1;                           // G7 flushed first: this move opens the new window
            if (pw >= P.K) {
                if (m > 0) { qmcd_flush_phase<MS>(P, s, cl, w, m); m = 0; }
                pw = 0;
            }
        }
        qmcd_writeback_M<MS>(P, s, w, m);
        if (r == 0 && tid == 0) { P.m[b] = m; if (QMCD_LOCKSTEP(P)) P.counters[(size_t)b * 8 + 7] = pw; }
        return;
    }

    if (A.mode == QMCD_MODE_FLUSH) {
        if (m > 0) qmcd_flush_phase<false>(P, s, cl, w, m);   // M is in global memory between launches
        else if (r == 0 && tid == 0) P.counters[(size_t)b * 8 + 7] = 0;
        return;
    }

    // ---- QMCD_MODE_SWEEP: the whole move loop, no host round trip, one cluster
    // barrier per move (inside the look-ahead); every CTA decides for itself.
    qmcd_load_state<MS>(P, s, w, m);
    // (the blocked look-ahead has its own entries, qmcd_kernel_sweep / qmcd_kernel_sweep_ls: the host
    // never launches this one with A.blocked set; the per-move loop below is correct for any input)
    const int len = w.khi - w.klo;
    const bool prof = (r == 0 && tid == 0);
    int pw = QMCD_LOCKSTEP(P) ? (int)__ldcg(P.counters + (size_t)b * 8 + 7) : 0;   // proposals in the window (lock-step)
    long long cy_la = 0, cy_acc = 0, c0 = prof ? clock64() : 0, c_start = c0;
    for (int t = 0; t < A.n_moves; ++t) {
        const int j = (A.j_begin + t) % P.N;
        const size_t tb = (size_t)t * P.batch + b;
        // decision input and next move's operands: get them moving towards L2 early
        double u = 0.0; unsigned char mk = 0;
        if (A.uniforms) u = A.uniforms[tb]; else mk = A.mask[tb];
        if (t + 1 < A.n_moves) {
            const int jn = (j + 1 == P.N) ? 0 : j + 1;
            for (int k = tid * 16; k < len; k += QMCD_THREADS * 16) {
                qmcd_prefetch_l2(A.v + (tb + P.batch) * P.N + w.klo + k);
                qmcd_prefetch_l2(w.B + (size_t)jn * P.N + w.klo + k);
            }
        }
        bool inq;
        double R = qmcd_lookahead<MS>(P, s, cl, w, j, m, A.v + tb * P.N, pbuf, &inq);
        if (prof) { const long long c1 = clock64(); cy_la += c1 - c0; c0 = c1; }
        bool acc;
        if (A.uniforms) { double pa = fmin(1.0, R * R); acc = u < pa; }
        else acc = mk != 0;
        if (acc && (R == 0.0 || !isfinite(R))) {
            if (r == 0 && tid == 0) qmcd_set_status(P, QMCD_DEV_ESINGULAR, b, t);
            acc = false;
        }
        if (r == 0 && tid == 0) {
            if (A.R_out) A.R_out[tb] = R;
            if (A.acc_out) A.acc_out[tb] = acc ? 1 : 0;
        }
        if (acc) m = qmcd_do_accept<MS>(P, s, cl, w, j, m, R, inq, pbuf);
        if (QMCD_LOCKSTEP(P)) {
            // every proposal takes a slot (a rejected one adds a zero column of U,
            // i.e. nothing), so the window closes after K proposals for every walker at once
            pw = (acc && inq) ? 1 : pw + 1;
            if (pw >= P.K) {
                if (m > 0) { qmcd_flush_phase<MS>(P, s, cl, w, m); m = 0; }
                pw = 0;
            }
        }
        if (prof) { const long long c1 = clock64(); cy_acc += c1 - c0; c0 = c1; }   // accept + flush (per-move path)
    }
    if (QMCD_LOCKSTEP(P) && r == 0 && tid == 0) P.counters[(size_t)b * 8 + 7] = pw;
    qmcd_writeback_M<MS>(P, s, w, m);
    if (prof) {
        long long* pc = P.counters + (size_t)b * 8;
        pc[2] += cy_la; pc[5] += cy_acc; pc[6] += clock64() - c_start;
    }
    if (r == 0 && tid == 0) { P.sj[b] = -1; P.m[b] = m; }
}

// Common prologue / epilogue of both entry points.  BLOCKED = true: the blocked sweep only (its
// own register allocation: the per-move look-ahead of the generic entry is not compiled in).
template <int BLOCKED>      // 0 generic, 1 blocked sweep, 2 blocked sweep in lock-step
__device__ __forceinline__ void qmcd_kernel_body(const QmcdArgs& A) {
    extern __shared__ __align__(1024) unsigned char qmcd_smem_raw[];
    const QmcdDev& P = A.P;
    cg::cluster_group cl = cg::this_cluster();
    const int S = P.S;
    const int r = (S > 1) ? (int)cl.block_rank() : 0;
    const int cidx = blockIdx.x / S;                 // cluster index
    const int b = cidx / P.G_act, g = cidx - b * P.G_act;
    const QmcdSmem s = qmcd_carve(qmcd_smem_raw, P.N, P.K, S, P.m_in_smem != 0);
    const QmcdWalker w = qmcd_walker(P, b, r, g, P.G_act);
    if (threadIdx.x == 0) s.iflag[8] = 0;
    __syncthreads();
    if (g > 0) { qmcd_helper_loop(P, s, cl, w); return; }
    if (BLOCKED) {
        int m = __ldcg(P.m + b);
        qmcd_load_state<true>(P, s, w, m);
        m = qmcd_sweep_blocked<BLOCKED == 2>(A, s, cl, w, m);
        qmcd_writeback_M<true>(P, s, w, m);
        if (r == 0 && threadIdx.x == 0) { P.sj[b] = -1; P.m[b] = m; }
    } else {
        if (P.m_in_smem) qmcd_run<true>(A, s, cl, w);
        else qmcd_run<false>(A, s, cl, w);
    }
    if (P.G_act > 1) {                               // release the helpers (every return path lands here)
        if (S > 1) cl.sync(); else __syncthreads();
        if (r == 0 && threadIdx.x == 0)
            qmcd_st_release(P.go + b, ((unsigned long long)P.launch_id << 32) | ((unsigned long long)QMCD_GO_EXIT << 12));
    }
}

__global__ void __launch_bounds__(QMCD_THREADS, 1) qmcd_kernel(const QmcdArgs A) { qmcd_kernel_body<0>(A); }
__global__ void __launch_bounds__(QMCD_THREADS, 1) qmcd_kernel_sweep(const QmcdArgs A) { qmcd_kernel_body<1>(A); }
__global__ void __launch_bounds__(QMCD_THREADS, 1) qmcd_kernel_sweep_ls(const QmcdArgs A) { qmcd_kernel_body<2>(A); }
