// qmcd_block.cuh -- blocked look-ahead for qmcd_sweep (pre-staged proposals): the per-move chain of a block of 16
// proposals (qmcd_blk_chain, shared with the super-blocks of qmcd_superblock.cuh, the default path) and the sweep loop
// in 16-proposal blocks with LDG / cp.async strips (qmcd_sweep_blocked: shapes the super-block ring does not take).
//
// Inside one window (between two flushes) the stale inverse B0 is fixed, so every
// quantity the look-ahead of Eq. 3 needs for the next L
// proposals t0..t0+L-1 is an entry of three small products over the long axis N:
//     P[tl][i]  = B0[j_tl,:] . C[i,:]      (L x m0)   -> p of move tl, queued part
//     Q[tl][i]  = W[i,:]     . v_tl        (L x m0)   -> q of move tl, queued part
//     D[sl][tl] = B0[j_sl,:] . v_tl        (L x L)    -> d = D[tl][tl]; p, q against
//                                                        moves accepted inside the block
// They are computed ONCE per block with DMMA (each CTA on its column slice),
// summed over the cluster by a reduce-scatter + all-gather through distributed
// shared memory (two cluster barriers per BLOCK instead of one per move), and the
// per-move chain (c = M q, r = M^T p, R, decision, bordering of M) then runs out
// of shared memory alone, replicated in every CTA.  The arithmetic per entry is
// the same dot product the per-call path computes; only the summation order
// differs.  Accepted moves are appended to the queue (C, W, J) at the block's end.
#pragma once
// (included by qmcd_kernel.cuh after qmcd_flush_phase is defined)

#define QMCD_TB 16              // proposals per block
#define QMCD_BLK_KC 64          // columns per staged chunk of the left operands
#define QMCD_BLK_LDA 72         // its row stride (== 8 mod 16 doubles)
#define QMCD_BLK_MAXU 5         // units (8-column output tiles) per warp: 2*ceil(K/8)+2 <= 40

__host__ __device__ inline int qmcd_blk_Kp(int K) { return (K + 7) & ~7; }
__host__ __device__ inline int qmcd_blk_RL(int K) { return 2 * qmcd_blk_Kp(K) + QMCD_TB; }
// As | recv[16][RL] | G[16][RL] | ub[16] | Rb[16] | Z[2][16][16] | Xm[Kp][16] | Ym[16][Kp] | Um[Kp][16]
// As = [2][32][LDA] (cp.async staging of the left operands)
__host__ __device__ inline size_t qmcd_blk_as_doubles() { return (size_t)2 * 32 * QMCD_BLK_LDA; }
__host__ __device__ inline size_t qmcd_blk_smem_bytes(int K) {
    return (qmcd_blk_as_doubles() + (size_t)2 * QMCD_TB * qmcd_blk_RL(K) + 32 + 2 * QMCD_TB * QMCD_TB + 3 * (size_t)QMCD_TB * qmcd_blk_Kp(K) + 8) * 8;
}

struct QmcdBlk {
    double* As;     // [2][32][LDA]  rows 0..15: B0[j_tl, chunk], rows 16..31: v_tl[chunk]
    double* recv;   // [S][RPO][RL]  partial strips of the rows this CTA reduces
    double* G;      // [16][RL]      reduced strips: P | Q | D
    double* Z;      // [2][16][16]   e_jt^T A_cur^-1 v_s of the block, ping-pong over accepted moves
    double* Xm;     // [Kp][16]      M0 Q^T
    double* Ym;     // [16][Kp]      P M0
    double* Um;     // [Kp][16]      X Zc^-1
    int* al;        // [16]          block index of the e-th accepted move
    double* ub;     // [16]          decision inputs of the block (uniform or mask as 0/1)
    double* Rb;     // [16]          ratios of the block (written to R_out at the block's end)
};

__device__ inline QmcdBlk qmcd_blk_carve(double* base, int K) {
    QmcdBlk x;
    const int RL = qmcd_blk_RL(K);
    x.As = base; base += qmcd_blk_as_doubles();
    x.recv = base; base += QMCD_TB * RL;
    x.G = base; base += QMCD_TB * RL;
    x.ub = base; base += 16;
    x.Rb = base; base += 16;
    x.Z = base; base += 2 * QMCD_TB * QMCD_TB;
    x.Xm = base; base += QMCD_TB * qmcd_blk_Kp(K);
    x.Ym = base; base += QMCD_TB * qmcd_blk_Kp(K);
    x.Um = base; base += QMCD_TB * qmcd_blk_Kp(K);
    x.al = reinterpret_cast<int*>(base);
    return x;
}

__device__ __forceinline__ double2 qmcd_ldcg128(const double* p) {
    double2 v;
    asm volatile("ld.global.cg.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p) : "memory");
    return v;
}

// Left operands of a block, staged chunk by chunk (64 columns): rows 0..15 = B0[j_tl, :],
// rows 16..31 = v_tl, tl < L (rows >= L are zeroed).  Thread t copies vector (t & 31) of rows
// (t >> 5) + 8 i, i < 4; the four source row pointers are computed once per block.
struct QmcdBlkSrc { const double* p[4]; };
__device__ __forceinline__ QmcdBlkSrc qmcd_blk_src(const QmcdArgs& A, const QmcdWalker& w, int t0, int L) {
    QmcdBlkSrc r;
    const QmcdDev& P = A.P;
    const int N = P.N;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int row = (threadIdx.x >> 5) + 8 * i, tl = row & 15;
        r.p[i] = nullptr;
        if (tl < L) {
            if (row < 16) { int j = A.j_begin + t0 + tl; j %= N; r.p[i] = w.B + (size_t)j * N + w.klo; }
            else r.p[i] = A.v + ((size_t)(t0 + tl) * P.batch + w.b) * N + w.klo;
        }
    }
    return r;
}
__device__ __forceinline__ void qmcd_blk_stage(double* dst, const QmcdBlkSrc& src, int kc, int cw) {
    const int c2 = (threadIdx.x & 31) * 2;
    if (c2 >= cw) return;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int row = (threadIdx.x >> 5) + 8 * i;
        double* d = dst + row * QMCD_BLK_LDA + c2;
        if (src.p[i]) qmcd_cp_async16(d, src.p[i] + kc * QMCD_BLK_KC + c2);
        else { d[0] = 0.0; d[1] = 0.0; }
    }
}

// Row pointer (at this CTA's column slice) of the RIGHT operand row `row` of unit u:
//   u <  nP      : C[u*8 + g]        (valid while < m0)
//   u < 2 nP     : W[(u-nP)*8 + g]   (valid while < m0)
//   else         : v_{t0 + (u-2nP)*8 + g}  (valid while < L)
__device__ __forceinline__ const double* qmcd_blk_right(const QmcdArgs& A, const QmcdWalker& w, int u, int nP,
                                                        int g, int m0, int t0, int L) {
    const int N = A.P.N;
    if (u < nP) { const int i = u * 8 + g; return (i < m0) ? w.C + (size_t)i * N + w.klo : nullptr; }
    if (u < 2 * nP) { const int i = (u - nP) * 8 + g; return (i < m0) ? w.W + (size_t)i * N + w.klo : nullptr; }
    const int tl = (u - 2 * nP) * 8 + g;
    return (tl < L) ? A.v + ((size_t)(t0 + tl) * A.P.batch + w.b) * N + w.klo : nullptr;
}

// Cluster-wide sum of the strips: acc[i][a] = this CTA's partial of unit wid + 8 i, row block a.
// Reduce-scatter + all-gather through distributed shared memory; on return every CTA holds G.
__device__ __forceinline__ void qmcd_blk_reduce(const QmcdDev& P, const QmcdBlk& x, cg::cluster_group& cl, const QmcdWalker& w,
                                             double (&acc)[QMCD_BLK_MAXU][2][2], int nu, int nP) {
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, g = lane >> 2, c = lane & 3;
    const int S = P.S, K = P.K, Kp = qmcd_blk_Kp(K), RL = qmcd_blk_RL(K);
    // ---- reduce-scatter: strip row `row` is summed by CTA (row % S); every CTA
    // sends its partial of that row to slot [my rank][row / S] of the owner's recv
    const int RPO = (QMCD_TB + S - 1) / S;
#pragma unroll
    for (int i = 0; i < QMCD_BLK_MAXU; ++i) {
        if (i < nu) {
            const int u = wid + 8 * i;
            const int off = (u < nP) ? u * 8 : (u < 2 * nP) ? Kp + (u - nP) * 8 : 2 * Kp + (u - 2 * nP) * 8;
#pragma unroll
            for (int a = 0; a < 2; ++a) {
                const int row = a * 8 + g;
                const int owner = row % S;
                double* rb = (S > 1) ? cl.map_shared_rank(x.recv, owner) : x.recv;
                *reinterpret_cast<double2*>(rb + ((size_t)w.r * RPO + row / S) * RL + off + 2 * c) =
                    make_double2(acc[i][a][0], acc[i][a][1]);
            }
        }
    }
    if (S > 1) cl.sync(); else __syncthreads();
    // ---- owner: sum the S partials in rank order, all-gather the result into every CTA's G
    {
        const int ncol = 2 * nP * 8 + QMCD_TB;            // active columns: P | Q | D
        for (int idx = tid; idx < RPO * ncol; idx += QMCD_THREADS) {
            const int rl = idx / ncol, ci = idx - rl * ncol;
            const int row = rl * S + w.r;
            if (row >= QMCD_TB) continue;
            const int col = (ci < nP * 8) ? ci : (ci < 2 * nP * 8) ? Kp + (ci - nP * 8) : 2 * Kp + (ci - 2 * nP * 8);
            double v = 0.0;
            for (int r = 0; r < S; ++r) v += x.recv[((size_t)r * RPO + rl) * RL + col];
            for (int q = 0; q < S; ++q) {
                double* gb = (S > 1) ? cl.map_shared_rank(x.G, q) : x.G;
                gb[(size_t)row * RL + col] = v;
            }
        }
    }
    if (S > 1) cl.sync(); else __syncthreads();
}

// ---------------------------------------------------------------------------
// G strips of one block: DMMA on this CTA's column slice, then the cluster-wide
// sum.  On return every CTA holds, for tl < 16:
//   G[tl][i]            = P[tl][i]   i < m0
//   G[tl][Kp + i]       = Q[tl][i]   i < m0
//   G[tl][2 Kp + sl]    = D[tl][sl] = B0[j_tl,:] . v_sl
// ---------------------------------------------------------------------------
__device__ __noinline__ void qmcd_blk_strips(const QmcdArgs& A, const QmcdSmem& s, const QmcdBlk& x, cg::cluster_group& cl,
                                const QmcdWalker& w, int t0, int L, int m0) {
    const QmcdDev& P = A.P;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, g = lane >> 2, c = lane & 3;
    const int len = w.khi - w.klo;
    const int nP = (m0 + 7) >> 3, U = 2 * nP + 2;
    const int nchunks = (len + QMCD_BLK_KC - 1) / QMCD_BLK_KC;
    // my units: u = wid, wid + 8, ...
    int nu = 0;
    const double* rp[QMCD_BLK_MAXU];
#pragma unroll
    for (int i = 0; i < QMCD_BLK_MAXU; ++i) {
        const int u = wid + 8 * i;
        rp[i] = nullptr;
        if (u < U) { nu = i + 1; rp[i] = qmcd_blk_right(A, w, u, nP, g, m0, t0, L); }
    }
    double acc[QMCD_BLK_MAXU][2][2];
#pragma unroll
    for (int i = 0; i < QMCD_BLK_MAXU; ++i) { acc[i][0][0] = acc[i][0][1] = acc[i][1][0] = acc[i][1][1] = 0.0; }

    const QmcdBlkSrc src = qmcd_blk_src(A, w, t0, L);
    qmcd_blk_stage(x.As, src, 0, min(QMCD_BLK_KC, len));
    qmcd_cp_async_commit();
    for (int kc = 0; kc < nchunks; ++kc) {
        const int cw = min(QMCD_BLK_KC, len - kc * QMCD_BLK_KC);
        if (kc + 1 < nchunks) {
            qmcd_blk_stage(x.As + ((kc + 1) & 1) * 32 * QMCD_BLK_LDA, src, kc + 1,
                           min(QMCD_BLK_KC, len - (kc + 1) * QMCD_BLK_KC));
            qmcd_cp_async_commit();
        }
        // right-operand fragments of this chunk for all my units: straight from L2
        // (each element is read once per CTA), issued before waiting for the stage
        const int nq = cw >> 3;
        const double* cur = x.As + (kc & 1) * 32 * QMCD_BLK_LDA + g * QMCD_BLK_LDA + 2 * c;
#pragma unroll
        for (int i = 0; i < QMCD_BLK_MAXU; ++i) {
            if (i < nu) {
                const int u = wid + 8 * i;
                const int left = (u >= nP && u < 2 * nP) ? 16 : 0;      // Q = V x W^T, else B0 rows
                double2 bv[8];
#pragma unroll
                for (int q = 0; q < 8; ++q)
                    bv[q] = (rp[i] != nullptr && q < nq) ? qmcd_ldcg128(rp[i] + kc * QMCD_BLK_KC + 8 * q + 2 * c)
                                                         : make_double2(0.0, 0.0);
                if (i == 0) {
                    if (kc + 1 < nchunks) qmcd_cp_async_wait<1>(); else qmcd_cp_async_wait<0>();
                    __syncthreads();
                }
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    if (q < nq) {
                        const double2 a0 = qmcd_lds128(cur + (left + 0) * QMCD_BLK_LDA + 8 * q);
                        const double2 a1 = qmcd_lds128(cur + (left + 8) * QMCD_BLK_LDA + 8 * q);
                        qmcd_dmma(acc[i][0][0], acc[i][0][1], a0.x, bv[q].x);
                        qmcd_dmma(acc[i][1][0], acc[i][1][1], a1.x, bv[q].x);
                        qmcd_dmma(acc[i][0][0], acc[i][0][1], a0.y, bv[q].y);
                        qmcd_dmma(acc[i][1][0], acc[i][1][1], a1.y, bv[q].y);
                    }
                }
            } else if (i == 0) {
                if (kc + 1 < nchunks) qmcd_cp_async_wait<1>(); else qmcd_cp_async_wait<0>();
                __syncthreads();
            }
        }
        __syncthreads();
    }

    qmcd_blk_reduce(P, x, cl, w, acc, nu, nP);
}

// X = M0 Q^T and Y = P M0 of one block with M in GLOBAL memory (K too large for a shared-memory copy): M0 is staged
// 16 rows at a time into the (idle) operand area x.As; thread (il, tl) forms X[p0 + il][tl], thread (t, bq) keeps
// Y[t][bq + 16 u] in registers over all panels.  Needs K even (16-byte row alignment) and K <= 16 * QMCD_BLK_YU.
#define QMCD_BLK_YU 10
__device__ __noinline__ void qmcd_blk_xy_global(const QmcdDev& P, const QmcdBlk& x, const QmcdWalker& w, int m0, int L, int RL) {
    const int tid = threadIdx.x, K = P.K, Kp = qmcd_blk_Kp(K), ldg = P.ldMg;
    const int ldp = Kp + 2, m0e = (m0 + 1) & ~1, vpr = m0e >> 1;
    double* Mp = x.As;
    const int t = tid >> 4, bq = tid & 15;
    double ya[QMCD_BLK_YU];
#pragma unroll
    for (int u = 0; u < QMCD_BLK_YU; ++u) ya[u] = 0.0;
    const double* Gq = x.G + (size_t)bq * RL + Kp;         // Q[tl = bq][:]  (X part: il = t, tl = bq)
    const double* Gp = x.G + (size_t)t * RL;               // P[t][:]        (Y part)
    for (int p0 = 0; p0 < m0; p0 += 16) {
        const int pr = min(16, m0 - p0);
        __syncthreads();                                   // the previous panel has been consumed
        for (int i0 = tid; i0 < pr * vpr; i0 += 4 * QMCD_THREADS) {
            double2 v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int idx = i0 + u * QMCD_THREADS;
                if (idx < pr * vpr) { const int r = idx / vpr, c2 = (idx - r * vpr) * 2; v[u] = qmcd_ldcg128(w.M + (size_t)(p0 + r) * ldg + c2); }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int idx = i0 + u * QMCD_THREADS;
                if (idx < pr * vpr) { const int r = idx / vpr, c2 = (idx - r * vpr) * 2; *reinterpret_cast<double2*>(Mp + r * ldp + c2) = v[u]; }
            }
        }
        __syncthreads();
        if (t < pr) {                                      // X[p0 + t][bq]
            double xa = 0.0;
            if (bq < L) { const double* row = Mp + t * ldp; for (int b = 0; b < m0; ++b) xa += row[b] * Gq[b]; }
            x.Xm[(p0 + t) * QMCD_TB + bq] = xa;
        }
        if (t < L) {
            for (int il = 0; il < pr; ++il) {
                const double pv = Gp[p0 + il];
                const double* row = Mp + il * ldp + bq;
#pragma unroll
                for (int u = 0; u < QMCD_BLK_YU; ++u) if (bq + 16 * u < m0) ya[u] += pv * row[16 * u];
            }
        }
    }
#pragma unroll
    for (int u = 0; u < QMCD_BLK_YU; ++u) if (bq + 16 * u < m0) x.Ym[t * Kp + bq + 16 * u] = ya[u];
}

// ---------------------------------------------------------------------------
// The per-move part of one block of L <= 16 proposals, from the reduced strips to the decisions
// and to M = S^-1 of the grown queue.  x.G (row stride RL) holds P at column 0, Q at Kp, D at
// 2 Kp; x.ub the decision inputs.  With M0 the inverse of S at the block's start,
//     Z[t][s] = D[t][s] - P[t,:] M0 Q[s,:]^T  =  e_{j_t}^T A_cur^-1 v_s     (t, s < L)
// is formed for ALL moves of the block at once; the ratio of move t is Z[t][t]
// (the Schur complement of the bordered S), and accepting move e
// applies the sweep operator on index e:
//     Z[i][j] -= Z[i][e] Z[e][j] / Z[e][e],  Z[e][j] /= Z[e][e],  Z[i][e] /= -Z[e][e],  Z[e][e] = 1/Z[e][e]
// -- one element per thread, one barrier per ACCEPTED move, nothing for a rejected
// one.  After the block the swept part of Z is Zc^-1 (Zc = Z0 on the accepted
// moves), and M = S^-1 for the grown queue follows from the block-bordering
// identity  M11 = M0 + X Zc^-1 Y,  M12 = -X Zc^-1,  M21 = -Zc^-1 Y,  M22 = Zc^-1
// with X = M0 Q_acc^T, Y = P_acc M0 (formed with Z0, in parallel, at the start).
// In exact arithmetic this is the move-by-move bordering of qmcd_accept_update.
// t = launch index of the block's first proposal, j0 = its electron.  Every CTA of the
// cluster runs this on the same numbers, so decisions agree without communication.
// Returns the mask of accepted moves (na of them): x.Rb holds the ratios, s.Js is extended.
// ---------------------------------------------------------------------------
template <bool MS>
__device__ __forceinline__ unsigned qmcd_blk_chain(const QmcdArgs& A, const QmcdSmem& s, const QmcdBlk& x, const QmcdWalker& w,
                                                   int RL, int t, int j0, int L, int m0, int& na_out) {
    const QmcdDev& P = A.P;
    const int tid = threadIdx.x;
    const int N = P.N, K = P.K, Kp = qmcd_blk_Kp(K), ldM = qmcd_ldM(K);
    // ---- X = M0 Q^T (Xm[i][t]) and Y = P M0 (Ym[t][b]) for every move of the block
    if (MS) {
        for (int idx = tid; idx < m0 * QMCD_TB; idx += QMCD_THREADS) {
            const int i = idx >> 4, tl = idx & 15;
            double xa = 0.0, ya = 0.0;
            if (tl < L) {
                const double* Gq = x.G + (size_t)tl * RL + Kp;      // Q[tl][:]
                const double* Gp = x.G + (size_t)tl * RL;           // P[tl][:]
                for (int b = 0; b < m0; ++b) {
                    xa += s.Ms[(size_t)i * ldM + b] * Gq[b];
                    ya += Gp[b] * s.Ms[(size_t)b * ldM + i];
                }
            }
            x.Xm[i * QMCD_TB + tl] = xa;
            x.Ym[tl * Kp + i] = ya;
        }
    } else {
        qmcd_blk_xy_global(P, x, w, m0, L, RL);
    }
    __syncthreads();
    // ---- Z0 = D - P X : one element per thread
    double* Zc = x.Z;                                  // current / next buffer (ping-pong)
    double* Zn = x.Z + QMCD_TB * QMCD_TB;
    {
        const int ti = tid >> 4, sj = tid & 15;
        double z = 0.0;
        if (ti < L && sj < L) {
            z = x.G[(size_t)ti * RL + 2 * Kp + sj];
            const double* Gp = x.G + (size_t)ti * RL;
            for (int i = 0; i < m0; ++i) z -= Gp[i] * x.Xm[i * QMCD_TB + sj];
        }
        Zc[tid] = z;
    }
    __syncthreads();
    unsigned accmask = 0;
    int na = 0;
    for (int tl = 0; tl < L; ++tl) {
        const double R = Zc[tl * QMCD_TB + tl];
        bool acc;
        if (A.uniforms) { const double pa = fmin(1.0, R * R); acc = x.ub[tl] < pa; }
        else acc = x.ub[tl] != 0.0;
        if (acc && (R == 0.0 || !isfinite(R))) {
            if (w.r == 0 && tid == 0) qmcd_set_status(P, QMCD_DEV_ESINGULAR, w.b, t + tl);
            acc = false;
        }
        if (tid == 0) x.Rb[tl] = R;
        if (acc) {
            // sweep operator on index tl: thread (i, jj) owns Z[i][jj]
            const int i = tid >> 4, jj = tid & 15;
            const double rp = 1.0 / R;
            const double zie = Zc[i * QMCD_TB + tl], zej = Zc[tl * QMCD_TB + jj], zij = Zc[tid];
            double zn;
            if (i == tl) zn = (jj == tl) ? rp : zej * rp;
            else zn = (jj == tl) ? -zie * rp : zij - zie * (zej * rp);
            Zn[tid] = zn;
            __syncthreads();
            double* tmp = Zc; Zc = Zn; Zn = tmp;
            accmask |= 1u << tl;
            na += 1;
        }
    }
    // ---- M for the grown queue (block bordering); al(e) = block index of the e-th accepted move
    if (na > 0) {
        int* al_s = x.al;
        if (tid < na) al_s[tid] = __fns(accmask, 0, tid + 1);
        __syncthreads();
        // U = X Zc^-1 restricted to accepted moves: U[i][f] = sum_e Xm[i][al_e] W1[e][f], W1 = Z[al_e][al_f]
        for (int idx = tid; idx < m0 * na; idx += QMCD_THREADS) {
            const int i = idx / na, f = idx - i * na;
            double u = 0.0;
            for (int e = 0; e < na; ++e) u += x.Xm[i * QMCD_TB + al_s[e]] * Zc[al_s[e] * QMCD_TB + al_s[f]];
            x.Um[i * QMCD_TB + f] = u;
        }
        __syncthreads();
        // M11 += U Y_acc ; M12 = -U ; M21 = -W1 Y_acc ; M22 = W1
        const int mn = m0 + na;
        auto newM = [&](int a, int b, double mold) -> double {
            double v;
            if (a < m0 && b < m0) {
                v = mold;
                for (int f = 0; f < na; ++f) v += x.Um[a * QMCD_TB + f] * x.Ym[al_s[f] * Kp + b];
            } else if (a < m0) {
                v = -x.Um[a * QMCD_TB + (b - m0)];
            } else if (b < m0) {
                v = 0.0;
                for (int f = 0; f < na; ++f) v -= Zc[al_s[a - m0] * QMCD_TB + al_s[f]] * x.Ym[al_s[f] * Kp + b];
            } else {
                v = Zc[al_s[a - m0] * QMCD_TB + al_s[b - m0]];
            }
            return v;
        };
        if (MS) {
            for (int idx = tid; idx < mn * mn; idx += QMCD_THREADS) {
                const int a = idx / mn, b = idx - a * mn;
                s.Ms[(size_t)a * ldM + b] = newM(a, b, (a < m0 && b < m0) ? s.Ms[(size_t)a * ldM + b] : 0.0);
            }
        } else if (w.r == 0) {
            // M in global memory (row stride P.ldMg), written by the leader CTA only; four elements per thread in flight
            const int ldg = P.ldMg;
            for (int i0 = tid; i0 < mn * mn; i0 += 4 * QMCD_THREADS) {
                double mo[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int idx = i0 + u * QMCD_THREADS;
                    const int a = idx / mn, b = idx - a * mn;
                    mo[u] = (idx < mn * mn && a < m0 && b < m0) ? __ldcg(w.M + (size_t)a * ldg + b) : 0.0;
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int idx = i0 + u * QMCD_THREADS;
                    if (idx < mn * mn) { const int a = idx / mn, b = idx - a * mn; w.M[(size_t)a * ldg + b] = newM(a, b, mo[u]); }
                }
            }
            __threadfence();
        }
        if (tid < na) s.Js[m0 + tid] = (j0 + al_s[tid]) % N;
    }
    na_out = na;
    return accmask;
}

// ---------------------------------------------------------------------------
// The sweep loop in blocks of 16 proposals, operands through LDG / cp.async (short column
// slices, K > 64; the super-block loop of qmcd_superblock.cuh serves the other shapes).
// Returns the queue length at the end.
// ---------------------------------------------------------------------------
// LS: the lock-step variant, a compile-time flag: a run-time test in this loop cost the
// default scheme 12 % on c1 (measured A/B on one box), so each reading has its own kernel entry.
template <bool LS, bool MS>
__device__ int qmcd_sweep_blocked(const QmcdArgs& A, const QmcdSmem& s, cg::cluster_group& cl,
                                  const QmcdWalker& w, int m) {
    const QmcdDev& P = A.P;
    const int tid = threadIdx.x;
    const int N = P.N, K = P.K, RL = qmcd_blk_RL(K);
    const int len = w.khi - w.klo;
    const QmcdBlk x = qmcd_blk_carve(s.rs, K);
    // cycle accounting by one thread of the leader CTA (every phase boundary is a barrier)
    const bool prof = (w.r == 0 && tid == 0);
    long long cy_la = 0, cy_chain = 0, cy_app = 0, cy_fl = 0, c0 = prof ? clock64() : 0, c_start = c0;
#define QMCD_TICK(acc_) do { if (prof) { const long long c1_ = clock64(); (acc_) += c1_ - c0; c0 = c1_; } } while (0)
    int t = 0;
    // lock-step: pw = proposals in the current window; a block never crosses its end
    int pw = LS ? (int)__ldcg(P.counters + (size_t)w.b * 8 + 7) : 0;
    while (t < A.n_moves) {
        const int j0 = (A.j_begin + t) % N;
        int L = min(min(QMCD_TB, LS ? min(K - pw, K - m) : K - m), A.n_moves - t);
        // an electron already queued may not be proposed inside a block (G7):
        // cut the block before it, or flush first when it is the block's first move
        {
            bool hit = false;
            for (int i = tid; i < m; i += QMCD_THREADS) { int dj = s.Js[i] - j0; if (dj < 0) dj += N; hit |= (dj < L); }
            if (__syncthreads_or(hit)) {
                if (tid == 0) {
                    int lh = L;
                    for (int i = 0; i < m; ++i) { int dj = s.Js[i] - j0; if (dj < 0) dj += N; lh = min(lh, dj); }
                    s.iflag[0] = lh;
                }
                __syncthreads();
                L = s.iflag[0];
                __syncthreads();
                if (L == 0) {
                    QMCD_TICK(cy_la);
                    qmcd_flush_phase<MS>(P, s, cl, w, m);
                    QMCD_TICK(cy_fl);
                    m = 0; pw = 0;
                    continue;
                }
            }
        }
        if (tid < L) {
            const size_t tb = (size_t)(t + tid) * P.batch + w.b;
            x.ub[tid] = A.uniforms ? A.uniforms[tb] : (A.mask[tb] ? 1.0 : 0.0);
        }
        // next block's operands: get them moving towards L2
        for (int idx = tid; idx < QMCD_TB * ((len + 15) >> 4); idx += QMCD_THREADS) {
            const int tl = idx / ((len + 15) >> 4), k = (idx - tl * ((len + 15) >> 4)) << 4;
            const int tn = t + L + tl;
            if (tn < A.n_moves) {
                qmcd_prefetch_l2(A.v + ((size_t)tn * P.batch + w.b) * N + w.klo + k);
                qmcd_prefetch_l2(w.B + (size_t)((A.j_begin + tn) % N) * N + w.klo + k);
            }
        }
        qmcd_blk_strips(A, s, x, cl, w, t, L, m);
        QMCD_TICK(cy_la);

        const int m0 = m;
        int na = 0;
        const unsigned accmask = qmcd_blk_chain<MS>(A, s, x, w, RL, t, j0, L, m0, na);
        QMCD_TICK(cy_chain);
        // ---- append the block's accepted moves to the queue: C[slot] = v, W[slot] = B0[j,:]
        {
            // four 16-byte vectors of each source row in flight per thread (the copy is a latency chain otherwise)
            const int vpr = len >> 1, total = na * vpr;
            for (int i0 = tid; i0 < total; i0 += 4 * QMCD_THREADS) {
                double2 vv[4], bb[4];
                size_t off[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int idx = i0 + u * QMCD_THREADS;
                    if (idx < total) {
                        const int e = idx / vpr, k = (idx - e * vpr) * 2;
                        const int al = __fns(accmask, 0, e + 1);
                        vv[u] = qmcd_ldcg128(A.v + ((size_t)(t + al) * P.batch + w.b) * N + w.klo + k);
                        bb[u] = qmcd_ldcg128(w.B + (size_t)((j0 + al) % N) * N + w.klo + k);
                        off[u] = (size_t)(m0 + e) * N + w.klo + k;
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    if (i0 + u * QMCD_THREADS < total) {
                        qmcd_stg128(w.C + off[u], vv[u].x, vv[u].y);
                        qmcd_stg128(w.W + off[u], bb[u].x, bb[u].y);
                    }
                }
            }
            __syncthreads();                       // Rb of the last move
            if (w.r == 0 && tid < L) {
                const size_t tb = (size_t)(t + tid) * P.batch + w.b;
                if (A.R_out) A.R_out[tb] = x.Rb[tid];
                if (A.acc_out) A.acc_out[tb] = (accmask >> tid) & 1u;
            }
            if (w.r == 0) {
                for (int e = tid; e < na; e += QMCD_THREADS) w.J[m0 + e] = (j0 + (int)__fns(accmask, 0, e + 1)) % N;
                if (tid == 0) P.counters[(size_t)w.b * 8 + 0] += na;
            }
        }
        m = m0 + na;
        t += L;
        __syncthreads();
        QMCD_TICK(cy_app);
        // flush when the queue is full -- or nearly full: a few moves early is neutral
        // and avoids a tail of 4-, 2-, 1-move blocks (several blocks per window at 50 % acceptance)
        if (LS) {
            pw += L;
            if (pw >= K) {                             // every walker closes its window here, rank m <= K
                if (m > 0) { qmcd_flush_phase<MS>(P, s, cl, w, m); m = 0; QMCD_TICK(cy_fl); }
                pw = 0;
            }
        } else if (K - m < max(1, min(QMCD_TB / 2, K / 4))) { qmcd_flush_phase<MS>(P, s, cl, w, m); m = 0; QMCD_TICK(cy_fl); }
    }
    if (LS && w.r == 0 && tid == 0) P.counters[(size_t)w.b * 8 + 7] = pw;
    if (prof) {
        long long* pc = P.counters + (size_t)w.b * 8;
        pc[2] += cy_la; pc[3] += cy_chain; pc[4] += cy_app; pc[5] += cy_fl; pc[6] += clock64() - c_start;
    }
#undef QMCD_TICK
    return m;
}
