// qmcd_kernel.cuh -- the __global__ entries over one body.  The grid is `batch` LEADER clusters of
// S CTAs (cluster b leads walker b: look-ahead, accept, and the posting of its flush jobs) followed,
// in qmcd_sweep / qmcd_flush launches, by the POOL: CTAs that lead no walker and take flush tiles of
// whichever walker has some (work stealing through one CAS per tile).  While one walker's leader
// runs its look-ahead chain, the pool and the other leaders keep the FP64 tensor pipe busy with the
// flushes of the others; every SM of the device is in the grid.
#pragma once
#include "qmcd_phases.cuh"
#include "qmcd_flush_mma.cuh"
#include "qmcd_flush_tma.cuh"

// ---- job words (QmcdDev::ticket / jdesc / fin), all at gpu scope
// jdesc = job number << 32 | ntiles << 16 | phase << 12 | m   (m <= 4095: checked by qmcd_create)
__device__ __forceinline__ unsigned long long qmcd_jdesc_pack(unsigned seq, int m, int phase, int ntiles) {
    return ((unsigned long long)seq << 32) | ((unsigned long long)(unsigned)ntiles << 16) |
           ((unsigned long long)(unsigned)phase << 12) | (unsigned long long)(unsigned)m;
}
// does the (ticket, descriptor) pair read by one thread name a job with a tile left?
__device__ __forceinline__ bool qmcd_job_has_tile(unsigned long long t, unsigned long long d) {
    return (t >> 32) != 0 && (t >> 32) == (d >> 32) && (unsigned)t < (unsigned)((d >> 16) & 0xFFFFu);
}
// Try to take one tile of walker b's posted job.  One thread.  Returns the tile (>= 0) and the
// job's (seq, m, phase), or -1 when the walker has no tile to give right now.  The descriptor is
// written before the ticket is released and carries the job number, so a pair that matches and
// survives the CAS belongs to one job.
__device__ __forceinline__ int qmcd_take_tile(const QmcdDev& P, int b, unsigned& seq, int& m, int& phase) {
    for (int tries = 0; tries < 4; ++tries) {
        const unsigned long long t = qmcd_ld_acquire(P.ticket + b);
        const unsigned long long d = __ldcg(P.jdesc + b);
        if (!qmcd_job_has_tile(t, d)) return -1;
        if (atomicCAS(P.ticket + b, t, t + 1) == t) {
            seq = (unsigned)(t >> 32); m = (int)(d & 0xFFFu); phase = (int)((d >> 12) & 0xFu);
            qmcd_fence_proxy_async();      // what the acquire made visible is read next through TMA (async proxy)
            return (int)(unsigned)t;
        }
    }
    return -1;
}
__device__ __forceinline__ void qmcd_tile_done(const QmcdDev& P, int b) {
    __syncthreads();                       // every thread's stores of the tile are issued
    if (threadIdx.x == 0) { __threadfence(); atomicAdd(P.fin + b, 1u); }
}

// One tile of a job, by all threads of this CTA: the TMA-fed kernel for the local K <= 64 phase
// (s.iflag[15] = iterations this CTA has pushed through the TMA ring), else the cp.async kernels.
__device__ void qmcd_do_tile(const QmcdDev& P, const QmcdSmem& s, int b, int phase, int m, int tile,
                             unsigned long long job_key, unsigned long long& mf_key) {
    if (P.use_tma && (phase == QMCD_JOB_LOCAL || phase == QMCD_JOB_ROWS_Y)) {
        unsigned char* base = reinterpret_cast<unsigned char*>(s.red);
        unsigned itc = (unsigned)s.iflag[15];
        const int key = qmcd_tma_NB(P.K) * 4 + (P.tile_rows == 128 ? 2 : 1);
        switch (key) {
            case 1 * 4 + 2: qmcd_flush_tile_tma<1, 2, false>(P, *s.tm, base, b, m, tile, itc); break;
            case 2 * 4 + 2: qmcd_flush_tile_tma<2, 2, false>(P, *s.tm, base, b, m, tile, itc); break;
            case 4 * 4 + 2: qmcd_flush_tile_tma<4, 2, false>(P, *s.tm, base, b, m, tile, itc); break;
            case 8 * 4 + 2: qmcd_flush_tile_tma<8, 2, false>(P, *s.tm, base, b, m, tile, itc); break;
            case 1 * 4 + 1: qmcd_flush_tile_tma<1, 1, false>(P, *s.tm, base, b, m, tile, itc); break;
            case 2 * 4 + 1: qmcd_flush_tile_tma<2, 1, false>(P, *s.tm, base, b, m, tile, itc); break;
            case 4 * 4 + 1: qmcd_flush_tile_tma<4, 1, false>(P, *s.tm, base, b, m, tile, itc); break;
            case 8 * 4 + 1: qmcd_flush_tile_tma<8, 1, false>(P, *s.tm, base, b, m, tile, itc); break;
            default: qmcd_flush_tile_tma<16, 1, true>(P, *s.tm, base, b, m, tile, itc); break;      // 64 < K <= 128, tile_rows 64
        }
        __syncthreads();                  // every warp has left the ring (and read iflag[15])
        if (threadIdx.x == 0) s.iflag[15] = (int)itc;
        mf_key = 0;
        return;
    }
    qmcd_flush_tile(P, s.dyn, b, phase, m, tile, job_key, mf_key);
}

// One job of walker b posted by its leader cluster: every CTA of the cluster takes tiles until none
// is left, then the leader thread waits until all `ntiles` are FINISHED (by whoever took them).
// s.iflag[8] = jobs posted so far in this launch, s.iflag[10] = tiles they had (same in every CTA).
__device__ void qmcd_run_job(const QmcdDev& P, const QmcdSmem& s, cg::cluster_group& cl,
                             const QmcdWalker& w, int m, int phase, unsigned long long& mf_key) {
    const int ntiles = qmcd_job_ntiles(P.N, P.tile_rows, phase);
    const int k = s.iflag[8] + 1;
    const unsigned expect = (unsigned)(s.iflag[10] + ntiles);
    if (w.r == 0 && threadIdx.x == 0) {
        __threadfence();                   // queue rows, M, J (and Y) written by this cluster, seen through its barriers
        P.jdesc[w.b] = qmcd_jdesc_pack((unsigned)k, m, phase, ntiles);
        qmcd_st_release(P.ticket + w.b, (unsigned long long)(unsigned)k << 32);
    }
    if (P.S > 1) cl.sync(); else __syncthreads();            // the job is posted before any CTA of the cluster looks for it
    const bool prof = threadIdx.x == 0 && blockIdx.x < QMCD_WSTAT_CTAS;
    long long c0 = prof ? clock64() : 0, ntile = 0;
    for (;;) {
        if (threadIdx.x == 0) {
            unsigned seq; int mm, ph;
            s.iflag[9] = qmcd_take_tile(P, w.b, seq, mm, ph);
        }
        __syncthreads();
        const int tile = s.iflag[9];
        __syncthreads();
        if (tile < 0) break;
        qmcd_do_tile(P, s, w.b, phase, m, tile, ((unsigned long long)(w.b + 1) << 32) | (unsigned)k, mf_key);
        qmcd_tile_done(P, w.b);
        ++ntile;
    }
    long long c1 = prof ? clock64() : 0;
    // (measured: letting the waiting leader take tiles of OTHER walkers' jobs delays its own look-ahead chain
    // by up to a tile time, so fewer jobs are posted and the pool starves: c4 0.74 -> 0.54, c3 unchanged)
    if (w.r == 0 && threadIdx.x == 0)
        while (qmcd_ld_acquire32(P.fin + w.b) != expect) __nanosleep(40);
    __syncthreads();
    if (prof) {                                              // leader CTAs: [2] = cycles waiting for tiles others took
        long long* ws = P.wstat + (size_t)blockIdx.x * 4;
        ws[0] += ntile; ws[1] += c1 - c0; ws[2] += clock64() - c1;
    }
    if (threadIdx.x == 0) { s.iflag[8] = k; s.iflag[10] = (int)expect; }
    if (P.S > 1) cl.sync(); else __syncthreads();
}

// Flush wrapper for the leader cluster: all its CTAs call it with the same m > 0.
// M goes back to global memory first (the flush reads it from there).
// Barriers: (entry) queue slots / M written by other CTAs are complete before the job is posted;
// (exit) nobody restages slot 0 or reads B rows before every tile is finished.
template <bool MS>
__device__ void qmcd_flush_phase(const QmcdDev& P, const QmcdSmem& s, cg::cluster_group& cl,
                                 const QmcdWalker& w, int m, bool writeback = true) {
    if (writeback) qmcd_writeback_M<MS>(P, s, w, m);
    if (P.use_tma && P.K <= 64 && qmcd_flush_use_mma(P)) qmcd_zero_pad_M(P, w, m);
    __threadfence();
    qmcd_fence_proxy_async();              // queue rows / M written above are read through TMA by the flush
    if (P.S > 1) cl.sync(); else __syncthreads();
    if (qmcd_flush_use_mma(P)) {
        unsigned long long mf_key = 0;     // the look-ahead arrays alias the flush's shared memory
        if (P.K <= 64) qmcd_run_job(P, s, cl, w, m, QMCD_JOB_LOCAL, mf_key);
        else {
            qmcd_run_job(P, s, cl, w, m, QMCD_JOB_Y, mf_key);
            qmcd_run_job(P, s, cl, w, m, QMCD_JOB_ROWS_Y, mf_key);
        }
    } else {
        qmcd_flush_simt(P, s, cl, w, m);   // CUDA-core path: the leader cluster alone, rows split over its CTAs
        if (P.S > 1) cl.sync(); else __syncthreads();
    }
    if (w.r == 0 && threadIdx.x == 0) {
        P.m[w.b] = 0;
        P.counters[(size_t)w.b * 8 + 1] += 1;
        P.counters[(size_t)w.b * 8 + 7] = 0;          // a new window starts (lock-step proposal count)
        P.fstat[(size_t)w.b * 2] += m;
    }
}

// Pool CTA: take tiles of any walker's posted job until every leader cluster has finished the launch.
// Warp 0 scans the ticket words (lane i looks at walker start + i), starting after the walker served last.
__device__ void qmcd_pool_loop(const QmcdDev& P, const QmcdSmem& s) {
    unsigned long long mf_key = 0;
    int start = (int)((blockIdx.x * 7u) % (unsigned)P.batch);
    const bool prof = threadIdx.x == 0 && blockIdx.x < QMCD_WSTAT_CTAS;
    long long cy_busy = 0, cy_seek = 0, ntile = 0, c_begin = prof ? clock64() : 0, c0 = c_begin;
    for (;;) {
        if (threadIdx.x < 32) {
            const int lane = threadIdx.x;
            int got = -1, gb = 0, gm = 0, gph = 0; unsigned gseq = 0;
            int idle = 0;
            for (;;) {
                for (int b0 = 0; b0 < P.batch && got < 0; b0 += 32) {
                    const int i = b0 + lane;
                    int bb = start + i; if (bb >= P.batch) bb -= P.batch;
                    bool has = false;
                    if (i < P.batch) {
                        const unsigned long long t = qmcd_ld_acquire(P.ticket + bb);
                        const unsigned long long d = __ldcg(P.jdesc + bb);
                        has = qmcd_job_has_tile(t, d);
                    }
                    unsigned mask = __ballot_sync(0xffffffffu, has);
                    while (mask != 0 && got < 0) {
                        const int l = __ffs(mask) - 1;
                        mask &= mask - 1;
                        int cand = start + b0 + l; if (cand >= P.batch) cand -= P.batch;
                        if (lane == 0) { got = qmcd_take_tile(P, cand, gseq, gm, gph); gb = cand; }
                        got = __shfl_sync(0xffffffffu, got, 0);
                    }
                }
                if (got >= 0) break;
                unsigned fin_leaders = 0;
                if (lane == 0) fin_leaders = qmcd_ld_acquire32(P.ctrl);
                fin_leaders = __shfl_sync(0xffffffffu, fin_leaders, 0);
                if (fin_leaders >= (unsigned)P.batch) { got = -2; break; }
                __nanosleep(idle < 8 ? 100 : 400);
                ++idle;
            }
            if (lane == 0) { s.iflag[9] = got; s.iflag[11] = gb; s.iflag[12] = gm; s.iflag[13] = gph; s.iflag[14] = (int)gseq; }
        }
        __syncthreads();
        const int tile = s.iflag[9], b = s.iflag[11], m = s.iflag[12], phase = s.iflag[13];
        const unsigned seq = (unsigned)s.iflag[14];
        __syncthreads();
        if (prof) { const long long c1 = clock64(); cy_seek += c1 - c0; c0 = c1; }
        if (tile < 0) break;
        qmcd_do_tile(P, s, b, phase, m, tile, ((unsigned long long)(b + 1) << 32) | seq, mf_key);
        qmcd_tile_done(P, b);
        if (prof) { const long long c1 = clock64(); cy_busy += c1 - c0; c0 = c1; ++ntile; }
        start = b;                          // stay with this walker while it has tiles (its M is staged here)
    }
    if (prof) {
        long long* ws = P.wstat + (size_t)blockIdx.x * 4;
        ws[0] += ntile; ws[1] += cy_busy; ws[2] += cy_seek; ws[3] += clock64() - c_begin;
    }
}

#include "qmcd_block.cuh"
#include "qmcd_superblock.cuh"

// Accept path shared by ACCEPT and SWEEP.  Called by ALL CTAs with the same
// (j, m, R, inq) and cf / rf valid in every CTA.  Returns the new m.
template <bool MS>
__device__ int qmcd_do_accept(const QmcdDev& P, const QmcdSmem& s, cg::cluster_group& cl,
                              const QmcdWalker& w, int j, int m, double R, bool inq, int& pbuf) {
    if (inq && P.slot_replace) {
        // repeated electron, slot replacement (G7, second alternative): no flush, m unchanged
        int a = 0;
        for (int i = 0; i < m; ++i) if (s.Js[i] == j) a = i;
        if (!MS && P.S > 1) cl.sync();
        qmcd_accept_replace<MS>(P, s, w, a, m, R);
        if (P.S > 1) cl.sync();        // slot a of C is complete before the next look-ahead reads it
        return m;
    }
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
        // every thread has read the staged proposal before the leader clears it
        if (S > 1) cl.sync(); else __syncthreads();
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
            if (inq && !P.slot_replace) pw = 1;        // G7 flushed first: this move opens the new window
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
            pw = (acc && inq && !P.slot_replace) ? 1 : pw + 1;
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

// Common prologue / epilogue of the entry points.  BLOCKED != 0: the blocked sweep only (its
// own register allocation: the per-move look-ahead of the generic entry is not compiled in).
template <int BLOCKED>      // 0 generic, 1 blocked sweep, 2 blocked sweep in lock-step, 3 blocked sweep with M in global memory
__device__ __forceinline__ void qmcd_kernel_body(const QmcdArgs& A, const QmcdTmaps& TM) {
    extern __shared__ __align__(1024) unsigned char qmcd_smem_raw[];
    const QmcdDev& P = A.P;
    cg::cluster_group cl = cg::this_cluster();
    const int S = P.S;
    const int r = (S > 1) ? (int)cl.block_rank() : 0;
    const int b = blockIdx.x / S;                    // cluster index: < batch leads walker b, else pool
    QmcdSmem s = qmcd_carve(qmcd_smem_raw, P.N, P.K, S, P.m_in_smem != 0);
    s.tm = &TM;
    if (threadIdx.x == 0) {
        s.iflag[8] = 0; s.iflag[10] = 0; s.iflag[12] = 0; s.iflag[13] = 0; s.iflag[14] = 0; s.iflag[15] = 0;
        if (P.use_tma) qmcd_tma_init_barriers(qmcd_smem_raw);
        if (P.la_tma) { qmcd_la_init_barriers(qmcd_smem_raw); qmcd_sb_app_init(qmcd_smem_raw); }
    }
    __syncthreads();
    if (b >= P.batch) { qmcd_pool_loop(P, s); return; }
    const QmcdWalker w = qmcd_walker(P, b, r);
    const long long c_launch = clock64();
    if (S > 1) cl.sync();                            // every CTA of the cluster runs before any remote shared-memory access
    if (BLOCKED == 3) {                              // blocked sweep with M in global memory (K too large for shared memory)
        int m = __ldcg(P.m + b);
        qmcd_load_state<false>(P, s, w, m);
        m = P.la_tma ? qmcd_sweep_sb<false, false>(A, s, cl, w, m) : qmcd_sweep_blocked<false, false>(A, s, cl, w, m);
        if (r == 0 && threadIdx.x == 0) { P.sj[b] = -1; P.m[b] = m; }
    } else if (BLOCKED) {
        int m = __ldcg(P.m + b);
        qmcd_load_state<true>(P, s, w, m);
        m = P.la_tma ? qmcd_sweep_sb<BLOCKED == 2, true>(A, s, cl, w, m) : qmcd_sweep_blocked<BLOCKED == 2, true>(A, s, cl, w, m);
        qmcd_writeback_M<true>(P, s, w, m);
        if (r == 0 && threadIdx.x == 0) { P.sj[b] = -1; P.m[b] = m; }
    } else {
        if (P.m_in_smem) qmcd_run<true>(A, s, cl, w);
        else qmcd_run<false>(A, s, cl, w);
    }
    if (threadIdx.x == 0 && blockIdx.x < QMCD_WSTAT_CTAS) P.wstat[(size_t)blockIdx.x * 4 + 3] += clock64() - c_launch;
    if (P.pool > 0) {                                // tell the pool this walker is done (every return path lands here)
        if (S > 1) cl.sync(); else __syncthreads();
        if (r == 0 && threadIdx.x == 0) { __threadfence(); atomicAdd(P.ctrl, 1u); }
    }
}

__global__ void __launch_bounds__(QMCD_THREADS, 1) qmcd_kernel(const QmcdArgs A, const __grid_constant__ QmcdTmaps TM) { qmcd_kernel_body<0>(A, TM); }
__global__ void __launch_bounds__(QMCD_THREADS, 1) qmcd_kernel_sweep(const QmcdArgs A, const __grid_constant__ QmcdTmaps TM) { qmcd_kernel_body<1>(A, TM); }
__global__ void __launch_bounds__(QMCD_THREADS, 1) qmcd_kernel_sweep_ls(const QmcdArgs A, const __grid_constant__ QmcdTmaps TM) { qmcd_kernel_body<2>(A, TM); }
__global__ void __launch_bounds__(QMCD_THREADS, 1) qmcd_kernel_sweep_gm(const QmcdArgs A, const __grid_constant__ QmcdTmaps TM) { qmcd_kernel_body<3>(A, TM); }
