// qmcd_superblock.cuh -- the look-ahead of qmcd_sweep in SUPER-BLOCKS, operands through a TMA ring (P.la_tma).
//
// Inside one window the stale inverse B0 is fixed and the proposals are pre-staged, so everything the look-ahead
// of Eq. 3 needs for the next nb <= 64 proposals t0 .. t0+nb-1 (electrons j0 .. j0+nb-1,
// none of them queued) is an entry of ONE product over the long axis N:
//
//     SBG = [ B0[j0.., :] . C^T  |  V[t0.., :] . W^T  |  B0[j0.., :] . V[t0.., :]^T ]      (shape x (m0 + m0 + shape))
//              P (vs the queue)     Q (vs the queue)      D (all pairs inside the super-block)
//
// with m0 the queue length at its start.  A move accepted INSIDE the super-block joins the queue with
// C[i,:] = v_a and W[i,:] = B0[j_a,:], so its column of P and Q for the later moves is a column / row of D: the
// 16-proposal blocks of the per-move chain (qmcd_blk_chain) gather their strips from SBG without touching memory
// again.  Against one strip pass per 16 proposals (qmcd_blk_strips) this reads every operand row ONCE per
// super-block (at 99 % acceptance and K = 64: 128 rows per window instead of 640), keeps all eight warps busy from
// m0 = 0 on (a 64 x 64 D is 32 output tiles), and fills the ring's pipeline once instead of four times.
// The rows of the accepted moves are appended to the queue at the super-block's end by bulk asynchronous copies.
//
// Ring stage (QMCD_SB_CW = 16 columns of this CTA's slice, 2 k-groups of 8):
//     B0[j0 ..][2][shape][8] | V[t0 ..][2][shape][8] | C[32 u ..][2][32][8] (u < ceil(m0/32)) | W likewise
// every box in the fragment-friendly k-major view of qmcd_flush_tma.cuh (8 x 8 fp64 blocks of 512 contiguous bytes:
// conflict-free 16-byte fragment loads).  shape = 16, 32 or 64 by the room left in the queue; a warp owns one block
// of 16 rows and up to QMCD_SB_MAXU output tiles of 16 x 8.
#pragma once
// (included by qmcd_kernel.cuh after qmcd_block.cuh)

#define QMCD_SB_MAXU 8          // output tiles (16 x 8) per warp
#define QMCD_SB_NS 3            // ring stages (== QMCD_LA_NS: the mbarriers of qmcd_la_init_barriers)
#define QMCD_SB_MAXR 16         // elements per thread in the cluster-wide sum
#define QMCD_SB_KMAX 128        // largest delay served (beyond it SBG, G, X, Y, U no longer fit beside the ring)
// k-groups of 8 columns per ring stage: 2 for K <= 64 (M in shared memory), 1 beyond (M in global memory; the stages
// hold up to 2 x 128 queue rows)
__host__ __device__ inline int qmcd_sb_nq(int K) { return K <= 64 ? 2 : 1; }

// largest queue length (rounded up to 8) a super-block of `shape` proposals may start at: 2 ceil(m0/8) + shape/8
// output-tile columns over 8 / (shape/16) warps per row block must stay <= QMCD_SB_MAXU per warp (shape 64: 32; 32: 112,
// kept at 56 for the size of a ring stage; 16: 248)
__host__ __device__ inline int qmcd_sb_m0p_max(int shape, int K) { return shape == 64 ? 32 : shape == 32 ? (K <= 64 ? 56 : 96) : 248; }
__host__ __device__ inline size_t qmcd_sb_stage_bytes(int K) {
    const int Kp = qmcd_blk_Kp(K);
    int rows = 0;
    for (int shape = 16; shape <= 64; shape *= 2) {
        const int mp = Kp < qmcd_sb_m0p_max(shape, K) ? Kp : qmcd_sb_m0p_max(shape, K);
        const int mb = (mp + 31) & ~31;            // C and W come in boxes of 32 rows
        if (2 * shape + 2 * mb > rows) rows = 2 * shape + 2 * mb;
    }
    return (size_t)rows * (qmcd_sb_nq(K) * 64);
}
__host__ __device__ inline size_t qmcd_sb_g_doubles(int K) {
    const int Kp = qmcd_blk_Kp(K);
    size_t n = 0;
    for (int shape = 16; shape <= 64; shape *= 2) {
        const int mp = Kp < qmcd_sb_m0p_max(shape, K) ? Kp : qmcd_sb_m0p_max(shape, K);
        const size_t v = (size_t)shape * (2 * mp + shape);
        if (v > n) n = v;
    }
    return n;
}
// row stride of the per-block strips x.G: odd, so that the 16 proposals of a block fall into different banks
__host__ __device__ inline int qmcd_sb_RL(int K) { return 2 * qmcd_blk_Kp(K) + QMCD_TB + 1; }
// ring | SBG | G[16][RL] | ub[16] | Rb[16] | Z[2][16][16] | Xm | Ym | Um | al[16] | alsb[64]
__host__ __device__ inline size_t qmcd_sb_smem_bytes(int K) {
    return QMCD_SB_NS * qmcd_sb_stage_bytes(K) +
           (qmcd_sb_g_doubles(K) + (size_t)QMCD_TB * qmcd_sb_RL(K) + 32 + 2 * QMCD_TB * QMCD_TB + 3 * (size_t)QMCD_TB * qmcd_blk_Kp(K) + 8 + 32) * 8;
}

struct QmcdSb {
    unsigned char* ring;
    double* SBG;
    int* alsb;      // [64] super-block index of the e-th move accepted in it
    QmcdBlk x;      // the chain's arrays (x.As = the ring: idle while the chain runs)
};
__device__ inline QmcdSb qmcd_sb_carve(double* base, int K) {
    QmcdSb b;
    b.ring = reinterpret_cast<unsigned char*>(base);
    base += QMCD_SB_NS * qmcd_sb_stage_bytes(K) / 8;
    b.SBG = base; base += qmcd_sb_g_doubles(K);
    QmcdBlk& x = b.x;
    x.As = reinterpret_cast<double*>(b.ring);
    x.recv = nullptr;
    x.G = base; base += (size_t)QMCD_TB * qmcd_sb_RL(K);
    x.ub = base; base += 16;
    x.Rb = base; base += 16;
    x.Z = base; base += 2 * QMCD_TB * QMCD_TB;
    x.Xm = base; base += QMCD_TB * qmcd_blk_Kp(K);
    x.Ym = base; base += QMCD_TB * qmcd_blk_Kp(K);
    x.Um = base; base += QMCD_TB * qmcd_blk_Kp(K);
    x.al = reinterpret_cast<int*>(base); base += 8;
    b.alsb = reinterpret_cast<int*>(base);
    return b;
}

// ---------------------------------------------------------------------------
// SBG of one super-block: DMMA on this CTA's column slice out of the TMA ring, then (S > 1) the cluster-wide sum in
// place.  On return every CTA holds, with nP = ceil(m0/8) and row stride ld = 8 (2 nP + shape/8), for a < shape:
//   SBG[a][i]              = B0[j0+a,:] . C[i,:]        i < m0
//   SBG[a][8 nP + i]       = V[t0+a,:]  . W[i,:]        i < m0
//   SBG[a][16 nP + s]      = B0[j0+a,:] . V[t0+s,:]     s < shape
// Rows of B0 past N and proposals past the launch are zero-filled by TMA; entries of rows / columns >= nb are never read.
// `itc` = chunks this CTA has pushed through the ring.
// ---------------------------------------------------------------------------
template <int NU, int NQ>     // NU output tiles per warp (tiles past the last one repeat the first and are dropped: the loop
                              // has no branch), NQ k-groups of 8 columns per stage
__device__ __noinline__ void qmcd_sb_strips(const QmcdArgs& A, const QmcdSmem& s, const QmcdSb& sb, cg::cluster_group& cl,
                                            const QmcdWalker& w, int t0, int j0, int shape, int m0, unsigned& itc) {
    constexpr int NS = QMCD_SB_NS;
    const QmcdDev& P = A.P;
    const QmcdTmaps& TM = *s.tm;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, g = lane >> 2, c = lane & 3;
    const int len = w.khi - w.klo, nch = len / (8 * NQ);
    const int nP = (m0 + 7) >> 3, nrb = shape >> 4, wpr = 8 / nrb;
    const int nQB = (nP + 3) >> 2;                              // 32-row boxes of C and of W (rows past m0: stale, finite, unused)
    const int ncu = 2 * nP + (shape >> 3), ld = 8 * ncu;
    const unsigned STAGE = (unsigned)qmcd_sb_stage_bytes(P.K);
    const unsigned stage_tx = (unsigned)NQ * (128u * shape + 4096u * nQB);
    const int si = shape == 64 ? 2 : shape == 32 ? 1 : 0;
    unsigned char* smem = reinterpret_cast<unsigned char*>(s.red);
    const unsigned bar0 = qmcd_su32(smem + QMCD_LA_BAR_OFF);
    const unsigned ring0 = qmcd_su32(sb.ring);
    const unsigned it0 = itc;
    const unsigned long long pol_keep = qmcd_policy_evict_last();
    auto issue = [&](int kc) {                    // one thread: the loads of chunk kc
        const unsigned gi = it0 + (unsigned)kc, st = gi % NS, u = gi / NS;
        if (u > 0) qmcd_mbar_wait(bar0 + 8 * NS + 8 * st, (u - 1) & 1);
        unsigned dst = ring0 + st * STAGE;
        const unsigned fb = bar0 + 8 * st;
        const int kg = (w.klo >> 3) + NQ * kc;
        qmcd_mbar_expect_tx(fb, stage_tx);
        qmcd_tma_load4(dst, &TM.Bs[si], 0, j0, kg, w.b, fb); dst += 64u * NQ * shape;
        qmcd_tma_load4(dst, &TM.Vs[si], 0, t0, kg, w.b, fb); dst += 64u * NQ * shape;
        for (int u32 = 0; u32 < nQB; ++u32) { qmcd_tma_load4_hint(dst, &TM.C32, 0, 32 * u32, kg, w.b, fb, pol_keep); dst += 2048 * NQ; }
        for (int u32 = 0; u32 < nQB; ++u32) { qmcd_tma_load4_hint(dst, &TM.W32, 0, 32 * u32, kg, w.b, fb, pol_keep); dst += 2048 * NQ; }
    };
    if (tid == 0) {
        for (int kc = 0; kc < NS - 1 && kc < nch; ++kc) issue(kc);
    }
    // this warp: row block rb, output-tile columns cu = wi + wpr i.  Stage layout in doubles: B0 rows [NQ][shape][8] at 0,
    // V rows at 8 NQ shape, C boxes [NQ][32][8] at 16 NQ shape, W boxes after them.  Right operand of tile column cu: BYTE
    // offset at k-group 0 (roff) and k-group stride (rqs); left operand: B0 rows (P, D) or V rows (Q: qs)
    const int rb = wid / wpr, wi = wid - rb * wpr;
    unsigned roff[NU], rqs[NU];
    bool qs[NU];
#pragma unroll
    for (int i = 0; i < NU; ++i) {
        int cu = wi + wpr * i;
        if (cu >= ncu) cu = wi;                                 // a tile this warp does not have: recompute its first one
        if (cu < nP) { roff[i] = 16 * NQ * shape + 256 * NQ * (cu >> 2) + ((cu & 3) * 8 + g) * 8 + 2 * c; rqs[i] = 256 * 8; qs[i] = false; }
        else if (cu < 2 * nP) { const int u8 = cu - nP; roff[i] = 16 * NQ * shape + 256 * NQ * nQB + 256 * NQ * (u8 >> 2) + ((u8 & 3) * 8 + g) * 8 + 2 * c; rqs[i] = 256 * 8; qs[i] = true; }
        else { const int d = cu - 2 * nP; roff[i] = 8 * NQ * shape + (d * 8 + g) * 8 + 2 * c; rqs[i] = 8 * shape * 8; qs[i] = false; }
        roff[i] *= 8;
    }
    double acc[NU][2][2];
#pragma unroll
    for (int i = 0; i < NU; ++i) { acc[i][0][0] = acc[i][0][1] = acc[i][1][0] = acc[i][1][1] = 0.0; }
    const unsigned loffB = (unsigned)((rb * 16 + g) * 8 + 2 * c) * 8u, qst = 64u * shape;   // bytes: B0 rows of my row block; next k-group
    for (int kc = 0; kc < nch; ++kc) {
        const unsigned gi = it0 + (unsigned)kc, st = gi % NS, u = gi / NS;
        const unsigned stg = ring0 + st * STAGE;
        qmcd_mbar_wait(bar0 + 8 * st, u & 1);
        if (wid == (kc & 7) && lane == 0 && kc + NS - 1 < nch) issue(kc + NS - 1);
        const unsigned Lb = stg + loffB, Lv = Lb + 64u * NQ * shape;    // rows 8..15 of the block at + 512 bytes
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            const double2 lb0 = qmcd_lds128s(Lb + q * qst), lb1 = qmcd_lds128s(Lb + q * qst + 512);
            const double2 lv0 = qmcd_lds128s(Lv + q * qst), lv1 = qmcd_lds128s(Lv + q * qst + 512);
            double2 bv[NU];
#pragma unroll
            for (int i = 0; i < NU; ++i) bv[i] = qmcd_lds128s(stg + roff[i] + q * rqs[i]);
            // all tiles' first k-step, then all tiles' second: dependent DMMAs are 2 NU issues apart
#pragma unroll
            for (int i = 0; i < NU; ++i) {
                qmcd_dmma(acc[i][0][0], acc[i][0][1], qs[i] ? lv0.x : lb0.x, bv[i].x);
                qmcd_dmma(acc[i][1][0], acc[i][1][1], qs[i] ? lv1.x : lb1.x, bv[i].x);
            }
#pragma unroll
            for (int i = 0; i < NU; ++i) {
                qmcd_dmma(acc[i][0][0], acc[i][0][1], qs[i] ? lv0.y : lb0.y, bv[i].y);
                qmcd_dmma(acc[i][1][0], acc[i][1][1], qs[i] ? lv1.y : lb1.y, bv[i].y);
            }
        }
        __syncwarp();
        if (lane == 0) qmcd_mbar_arrive(bar0 + 8 * NS + 8 * st);
    }
    itc = it0 + (unsigned)nch;
    // this CTA's partial sums
#pragma unroll
    for (int i = 0; i < NU; ++i) {
        const int cu = wi + wpr * i;
        if (cu < ncu) {
#pragma unroll
            for (int a = 0; a < 2; ++a)
                *reinterpret_cast<double2*>(sb.SBG + (size_t)(rb * 16 + a * 8 + g) * ld + cu * 8 + 2 * c) = make_double2(acc[i][a][0], acc[i][a][1]);
        }
    }
    const int S = P.S;
    if (S == 1) { __syncthreads(); return; }
    // cluster-wide sum in place: CTA r sums share r of the elements over the S partial copies (in rank order), holds the
    // sums in registers across the barrier after which nobody reads partials any more, and writes them to every copy
    cl.sync();
    {
        const int tot = shape * ld, per = (tot + S - 1) / S, lo = w.r * per, hi = min(tot, lo + per);
        double sm[QMCD_SB_MAXR];
#pragma unroll
        for (int k = 0; k < QMCD_SB_MAXR; ++k) {
            const int idx = lo + tid + k * QMCD_THREADS;
            sm[k] = 0.0;
            if (idx < hi) { double v = 0.0; for (int q = 0; q < S; ++q) v += cl.map_shared_rank(sb.SBG, q)[idx]; sm[k] = v; }
        }
        cl.sync();
#pragma unroll
        for (int k = 0; k < QMCD_SB_MAXR; ++k) {
            const int idx = lo + tid + k * QMCD_THREADS;
            if (idx < hi) for (int q = 0; q < S; ++q) cl.map_shared_rank(sb.SBG, q)[idx] = sm[k];
        }
        cl.sync();
    }
}

// Queue append of a super-block's accepted moves by bulk asynchronous copies: rows v -> C[slot] and B0[j,:] -> W[slot]
// (this CTA's column slice of each, in pieces of <= 8 KB) bounce through shared memory: the ring, SBG and the chain's
// arrays are all dead at this point.  Lane 0 of every warp copies the pieces wid, wid + 8, ... through two slots of its
// own (load k+1 in flight while piece k is stored): 16 slots per CTA, the issue cost spread over the warps -- the copy
// is bound by bytes in flight per SM and, for short rows, by instructions per piece.  All threads call; the caller
// barriers afterwards.  Header ints at QMCD_SB_APP_PH_OFF: loads each slot's mbarrier has completed.
#define QMCD_SB_APP_SLOTS 16
#define QMCD_SB_APP_BAR_OFF 640              // 16 mbarriers in the shared-memory header
#define QMCD_SB_APP_PH_OFF 384               // 16 ints in the shared-memory header
__device__ __forceinline__ void qmcd_sb_app_init(unsigned char* smem) {
    for (int i = 0; i < QMCD_SB_APP_SLOTS; ++i) {
        qmcd_mbar_init(qmcd_su32(smem + QMCD_SB_APP_BAR_OFF) + 8 * i, 1);
        reinterpret_cast<int*>(smem + QMCD_SB_APP_PH_OFF)[i] = 0;
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __noinline__ void qmcd_sb_append(const QmcdArgs& A, const QmcdSmem& s, const QmcdSb& sb, const QmcdWalker& w,
                                            int t0, int j0, int m0, int na) {
    if ((threadIdx.x & 31) != 0) return;
    const QmcdDev& P = A.P;
    const int N = P.N, len = w.khi - w.klo, wid = threadIdx.x >> 5;
    unsigned char* smem = reinterpret_cast<unsigned char*>(s.red);
    const unsigned rowbytes = (unsigned)len * 8u;
    const unsigned bounce = (unsigned)(reinterpret_cast<unsigned char*>(sb.x.al) - sb.ring) & ~127u;
    unsigned cap = (bounce / QMCD_SB_APP_SLOTS) & ~127u;               // bytes per slot
    if (cap > 8192u) cap = 8192u;
    const unsigned ppr = (rowbytes + cap - 1) / cap;                   // pieces per row
    const unsigned piece = (((rowbytes + ppr - 1) / ppr) + 15u) & ~15u;  // bytes per piece (the last one may be shorter)
    const int njobs = 2 * na * (int)ppr;
    const unsigned bar = qmcd_su32(smem + QMCD_SB_APP_BAR_OFF) + 16u * wid;
    int* ph = reinterpret_cast<int*>(smem + QMCD_SB_APP_PH_OFF) + 2 * wid;
    const unsigned slot0 = qmcd_su32(sb.ring) + (unsigned)(2 * wid) * cap;
    // job -> (source, destination, bytes): job = (e * 2 + which) * ppr + piece index
    auto job = [&](int jb, const double*& src, double*& dst, unsigned& bytes) {
        const int pi = jb % (int)ppr, r = jb / (int)ppr, e = r >> 1;
        const int a = sb.alsb[e];
        const unsigned off = (unsigned)pi * piece;
        bytes = min(piece, rowbytes - off);
        const size_t col = (size_t)w.klo + off / 8;
        src = (r & 1) ? w.B + (size_t)((j0 + a) % N) * N + col : A.v + ((size_t)(t0 + a) * P.batch + w.b) * N + col;
        dst = ((r & 1) ? w.W : w.C) + (size_t)(m0 + e) * N + col;
    };
    auto load = [&](int k) {                  // my k-th piece into slot k & 1
        const double* sp; double* dp; unsigned by; job(wid + 8 * k, sp, dp, by);
        qmcd_mbar_expect_tx(bar + 8 * (k & 1), by);
        qmcd_bulk_load(slot0 + (unsigned)(k & 1) * cap, sp, by, bar + 8 * (k & 1));
    };
    const int nk = (njobs - wid + 7) / 8;     // pieces of this warp
    if (nk <= 0) return;
    load(0);
    if (nk > 1) load(1);
    for (int k = 0; k < nk; ++k) {
        const int sl = k & 1;
        qmcd_mbar_wait(bar + 8 * sl, (unsigned)ph[sl] & 1u);
        ph[sl] += 1;
        const double* sp; double* dp; unsigned by; job(wid + 8 * k, sp, dp, by);
        qmcd_bulk_store(dp, slot0 + (unsigned)sl * cap, by);
        qmcd_bulk_commit();
        if (k + 2 < nk) { qmcd_bulk_wait_read0(); load(k + 2); }      // the slot has been read: the next piece may land in it
    }
    qmcd_bulk_wait0();                      // the rows are written before the caller's barrier
}

// ---------------------------------------------------------------------------
// The sweep loop in super-blocks (M in shared memory, replicated in every CTA of the cluster).  Returns the queue
// length at the end.  LS: the lock-step variant, a compile-time flag as in qmcd_sweep_blocked.
// ---------------------------------------------------------------------------
template <bool LS, bool MS>
__device__ int qmcd_sweep_sb(const QmcdArgs& A, const QmcdSmem& s, cg::cluster_group& cl, const QmcdWalker& w, int m) {
    constexpr int NQ = MS ? 2 : 1;                 // the host pairs M in shared memory with K <= 64 (qmcd_sb_nq)
    const QmcdDev& P = A.P;
    const int tid = threadIdx.x;
    const int N = P.N, K = P.K, Kp = qmcd_blk_Kp(K), RL = qmcd_sb_RL(K);
    const QmcdSb sb = qmcd_sb_carve(s.rs, K);
    const QmcdBlk& x = sb.x;
    const bool prof = (w.r == 0 && tid == 0);
    long long cy_la = 0, cy_chain = 0, cy_app = 0, cy_fl = 0, c0 = prof ? clock64() : 0, c_start = c0;
#define QMCD_TICK(acc_) do { if (prof) { const long long c1_ = clock64(); (acc_) += c1_ - c0; c0 = c1_; } } while (0)
    const int thresh = max(1, min(QMCD_TB / 2, K / 4));
    int t = 0, n_prop = 0, n_acc = 0;                                    // proposals decided / accepted so far in this launch
    // Stagger: walkers that start a launch together with empty queues would post their flush jobs in the same instant, window
    // after window (their timing is identical), and the pool would idle during the look-aheads in between.  The FIRST window of
    // walker b is therefore cut short to K (b mod G + 1) / G moves -- flushing early is neutral -- which spreads the
    // walkers' phases over the cycle; the later windows take K moves.  Not in lock-step (the windows are the proposals').
    int kcap = K;
    if (!LS && P.stagger && m == 0 && A.n_moves >= 2 * K) {
        const int G = min(P.batch, 8);
        kcap = max(1, K * ((w.b % G) + 1) / G);
    }
    int pw = LS ? (int)__ldcg(P.counters + (size_t)w.b * 8 + 7) : 0;     // lock-step: proposals in the current window
    while (t < A.n_moves) {
        const int j0 = (A.j_begin + t) % N;
        // proposals to look ahead: what the queue still takes (rounded up to whole blocks), not past the launch, the
        // wrap-around of the electron index (the rows of B0 are one box) or, lock-step, the window's end
        // (at the acceptance rate seen so far in this launch: a queue with room for 32 takes 64 proposals at 50 %; moves
        // beyond what the queue takes are looked at again by the next super-block)
        int nb = kcap - m;
        if (n_acc < n_prop) {                          // (nothing accepted yet: as long as allowed; never shorter than the room itself)
            const long long want = (n_acc > 0) ? ((long long)nb * n_prop + n_acc - 1) / n_acc : 64;
            nb = (int)min((long long)64, max((long long)nb, want));
        }
        nb = min(64, (nb + QMCD_TB - 1) & ~(QMCD_TB - 1));
        nb = min(nb, min(A.n_moves - t, N - j0));
        if (LS) nb = min(nb, K - pw);
        // an electron already queued may not be proposed inside a super-block (G7): cut before it, or flush
        // first when it is the first move
        {
            bool hit = false;
            for (int i = tid; i < m; i += QMCD_THREADS) { int dj = s.Js[i] - j0; if (dj < 0) dj += N; hit |= (dj < nb); }
            if (__syncthreads_or(hit)) {
                if (tid == 0) {
                    int lh = nb;
                    for (int i = 0; i < m; ++i) { int dj = s.Js[i] - j0; if (dj < 0) dj += N; lh = min(lh, dj); }
                    s.iflag[0] = lh;
                }
                __syncthreads();
                nb = s.iflag[0];
                __syncthreads();
                if (nb == 0) {
                    QMCD_TICK(cy_la);
                    qmcd_flush_phase<MS>(P, s, cl, w, m);
                    QMCD_TICK(cy_fl);
                    m = 0; pw = 0; kcap = K;
                    continue;
                }
            }
        }
        const int m0sb = m, nP = (m + 7) >> 3;
        int shape = nb > 32 ? 64 : nb > 16 ? 32 : 16;
        while (shape > 16 && 8 * nP > qmcd_sb_m0p_max(shape, K)) shape >>= 1;
        nb = min(nb, shape);
        const int ld = 8 * (2 * nP + (shape >> 3));
        {
            unsigned itc = (unsigned)s.iflag[12];
            const int nu = (2 * nP + (shape >> 3) + (128 / shape) - 1) / (128 / shape);     // output tiles per warp
            if (nu <= 2) qmcd_sb_strips<2, NQ>(A, s, sb, cl, w, t, j0, shape, m, itc);
            else if (nu <= 4) qmcd_sb_strips<4, NQ>(A, s, sb, cl, w, t, j0, shape, m, itc);
            else if (nu <= 6) qmcd_sb_strips<6, NQ>(A, s, sb, cl, w, t, j0, shape, m, itc);
            else qmcd_sb_strips<QMCD_SB_MAXU, NQ>(A, s, sb, cl, w, t, j0, shape, m, itc);
            if (tid == 0) s.iflag[12] = (int)itc;      // (read again only after the barriers below)
        }
        QMCD_TICK(cy_la);

        int o = 0, na_sb = 0;
        while (o < nb) {
            const int L = min(min(QMCD_TB, nb - o), kcap - m);
            if (tid < L) {
                const size_t tb = (size_t)(t + o + tid) * P.batch + w.b;
                x.ub[tid] = A.uniforms ? A.uniforms[tb] : (A.mask[tb] ? 1.0 : 0.0);
            }
            // the block's strips: queue entries from before the super-block out of P and Q, those accepted inside it out of D
            {
                const int wd = 2 * m + QMCD_TB;
                for (int idx = tid; idx < QMCD_TB * wd; idx += QMCD_THREADS) {
                    const int tl = idx / wd, ci = idx - tl * wd;
                    const double* row = sb.SBG + (size_t)(o + tl) * ld;
                    double v; int dst;
                    if (ci < m) { v = (ci < m0sb) ? row[ci] : row[16 * nP + sb.alsb[ci - m0sb]]; dst = ci; }
                    else if (ci < 2 * m) {
                        const int i = ci - m;
                        v = (i < m0sb) ? row[8 * nP + i] : sb.SBG[(size_t)sb.alsb[i - m0sb] * ld + 16 * nP + o + tl];
                        dst = Kp + i;
                    } else { const int sl = ci - 2 * m; v = row[16 * nP + o + sl]; dst = 2 * Kp + sl; }
                    x.G[(size_t)tl * RL + dst] = v;
                }
            }
            __syncthreads();
            int na = 0;
            const unsigned accmask = qmcd_blk_chain<MS>(A, s, x, w, RL, t + o, j0 + o, L, m, na);
            if (tid < na) sb.alsb[na_sb + tid] = o + x.al[tid];
            // M in global memory is written by the leader CTA alone: the others read it again in the next block
            if (!MS && P.S > 1) cl.sync(); else __syncthreads();   // (and: Rb of the last move, alsb)
            if (w.r == 0 && tid < L) {
                const size_t tb = (size_t)(t + o + tid) * P.batch + w.b;
                if (A.R_out) A.R_out[tb] = x.Rb[tid];
                if (A.acc_out) A.acc_out[tb] = (accmask >> tid) & 1u;
            }
            if (w.r == 0) {
                if (tid < na) w.J[m + tid] = (j0 + sb.alsb[na_sb + tid]) % N;
                if (tid == 0) P.counters[(size_t)w.b * 8 + 0] += na;
            }
            m += na; na_sb += na; o += L;
            n_prop += L; n_acc += na;
            QMCD_TICK(cy_chain);
            if (LS) { pw += L; if (pw >= K) break; }
            else if (kcap - m < thresh) break;
        }
        // ---- append the super-block's accepted moves to the queue: C[slot] = v, W[slot] = B0[j,:]
        if (na_sb > 0) qmcd_sb_append(A, s, sb, w, t, j0, m0sb, na_sb);
        __syncthreads();
        t += o;
        QMCD_TICK(cy_app);
        // flush when the queue is full -- or nearly full: a few moves early is neutral
        if (LS) {
            if (pw >= K) {                             // every walker closes its window here, rank m <= K
                if (m > 0) { qmcd_flush_phase<MS>(P, s, cl, w, m); m = 0; QMCD_TICK(cy_fl); }
                pw = 0;
            }
        } else if (kcap - m < thresh) {                // (m == 0: a shortened first window in which nothing was accepted)
            if (m > 0) { qmcd_flush_phase<MS>(P, s, cl, w, m); m = 0; QMCD_TICK(cy_fl); }
            kcap = K;
        }
    }
    if (LS && w.r == 0 && tid == 0) P.counters[(size_t)w.b * 8 + 7] = pw;
    if (prof) {
        long long* pc = P.counters + (size_t)w.b * 8;
        pc[2] += cy_la; pc[3] += cy_chain; pc[4] += cy_app; pc[5] += cy_fl; pc[6] += clock64() - c_start;
    }
#undef QMCD_TICK
    return m;
}
