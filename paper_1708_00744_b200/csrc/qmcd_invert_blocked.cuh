// qmcd_invert_blocked.cuh -- batched on-device inversion as a BLOCKED Gauss-Jordan
// elimination with partial (row) pivoting: the same arithmetic as qmcd_invert.cuh, step for step, but the
// elimination of KB <= 16 consecutive pivot columns is applied to the rest of the matrix in ONE pass, so the
// matrix crosses HBM N/KB times instead of N times (16 N^3 / KB bytes per walker).
//
// Walker b is owned by C CTAs, CTA c holding the row slots i == c (mod C).  Per panel of kb pivot columns [k0, k0+kb):
//   panel phase (ONE grid barrier per pivot step; only the N x kb panel columns, held in the owners' shared memory):
//     step s (k = k0 + s): every CTA publishes its candidate (largest |x_i[k]|, i >= k) with that row's panel entries
//     and multipliers, and the owner of slot k publishes slot k's; after the barrier all CTAs pick the same pivot slot p,
//     form the scaled pivot row's panel part rho_s, and eliminate column k from the panel entries of their own slots,
//     recording the multiplier f_i^(s).  Slot k takes the pivot row (multipliers so far -> row s of L, then cleared);
//     slot p takes old row k.  The other columns of rows k and p are swapped in place, a column segment per CTA.
//   phase A (non-pivot slots, other columns, chunk by chunk): rho_s[q] = (x_k0+s[q] - sum_{t<s} L[s][t] rho_t[q]) d_s is
//     rebuilt per chunk in shared memory from the (still untouched) pivot rows, then x_i[q] -= sum_s f_i^(s) rho_s[q].
//   phase B (the kb pivot slots, chunks dealt over the walker's CTAs): x_k0+s[q] = rho_s[q] - sum_{t>s} f_k0+s^(t) rho_t[q].
// In-place inverse: the pivot column entry of a row is cleared before its elimination (x[k] := -f d), so the panel
// columns hold the new inverse columns afterwards and are ordinary columns for the later panels.  The row swaps are
// undone at the end as one column gather per row, as in qmcd_invert.cuh.
#pragma once
#include "qmcd_invert.cuh"

#define QMCD_INVB_KB 16         // largest panel width
#define QMCD_INVB_REC (2 + 2 * QMCD_INVB_KB)   // doubles per candidate record: |value|, slot, panel entries, multipliers

struct QmcdInvBArgs {
    int N, batch, C, KB, CH;    // CH = columns per chunk of the passes
    const double* A;            // [batch][N][N] row-major
    double* X;                  // [batch][N][N] result (may alias A)
    int* piv;                   // [batch][N]    pivot slot of every step
    double* cand;               // [batch][2][C][REC]  candidate records, double-buffered by step parity
    double* kdat;               // [batch][2][2 KB]    slot k's panel entries and multipliers, by step parity
    double* lf;                 // [batch][KB][KB]     L (below the diagonal), d (diagonal), later multipliers of the pivot slots (above)
    int* info;                  // [batch] 0, or k+1 of the first zero / non-finite pivot
};

// is candidate (|value| v, slot i) a better pivot than (bv, bi)?  Largest modulus, lowest slot on ties; a NaN beats any
// number (it is then reported as a singular pivot).  A total order: every CTA picks the same pivot whatever the scan order.
__device__ __forceinline__ bool qmcd_invb_better(double v, int i, double bv, int bi) {
    if (i < 0) return false;
    if (bi < 0) return true;
    const bool vn = (v != v), bn = (bv != bv);
    if (vn != bn) return vn;
    if (vn) return i < bi;
    return v > bv || (v == bv && i < bi);
}

__host__ __device__ inline size_t qmcd_invb_smem_bytes(int N, int C, int KB, int CH) {
    const size_t SL = (size_t)(N + C - 1) / C;
    size_t a = ((size_t)KB * CH + 2 * SL * KB + 4 * QMCD_INVB_KB + 64) * 8;
    const size_t g = (size_t)N * 12 + 64;                    // the final gather: one row + the column map
    return a > g ? a : g;
}

__global__ void __launch_bounds__(QMCD_INV_THREADS, 1) qmcd_invert_blocked_kernel(const QmcdInvBArgs a) {
    namespace cg = cooperative_groups;
    extern __shared__ __align__(16) unsigned char invb_smem[];
    cg::grid_group grid = cg::this_grid();
    const int N = a.N, C = a.C, KB = a.KB, CH = a.CH;
    const int b = blockIdx.x / C, c = blockIdx.x - b * C;
    const int NT = (int)blockDim.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, NW = NT >> 5;
    const int SL = (N + C - 1) / C, nown = (N - c + C - 1) / C;       // slots per CTA (max / mine): slot i = c + C j
    double* rho = reinterpret_cast<double*>(invb_smem);                // [KB][CH]
    double* Xp = rho + (size_t)KB * CH;                                // [KB][SL] panel entries of my slots
    double* Fo = Xp + (size_t)SL * KB;                                 // [KB][SL] multipliers of my slots in this panel
    double* pe = Fo + (size_t)SL * KB;                                 // [KB] pivot row: panel entries -> rho_s (panel part)
    double* pf = pe + QMCD_INVB_KB;                                    // [KB] pivot row: multipliers so far
    double* ke = pf + QMCD_INVB_KB;                                    // [KB] old row k: panel entries
    double* kf = ke + QMCD_INVB_KB;                                    // [KB] old row k: multipliers
    __shared__ double s_val[QMCD_INV_THREADS / 32];
    __shared__ int s_idx[QMCD_INV_THREADS / 32];
    __shared__ int s_p, s_q;
    const double* Ab = a.A + (size_t)b * N * N;
    double* X = a.X + (size_t)b * N * N;
    double* cand = a.cand + (size_t)b * 2 * C * QMCD_INVB_REC;
    double* kdat = a.kdat + (size_t)b * 2 * 2 * QMCD_INVB_KB;
    double* lf = a.lf + (size_t)b * QMCD_INVB_KB * QMCD_INVB_KB;
    int* piv = a.piv + (size_t)b * N;
    const bool vec = ((N & 1) == 0) && ((reinterpret_cast<uintptr_t>(X) & 15) == 0) && ((CH & 1) == 0);

    for (int j = warp; j < nown; j += NW) {                            // copy my rows
        const size_t o = (size_t)(c + C * j) * N;
        for (int q = lane; q < N; q += 32) X[o + q] = Ab[o + q];
    }
    __syncthreads();
    for (int k0 = 0; k0 < N; k0 += KB) {
        const int kb = min(KB, N - k0);
        for (int idx = tid; idx < nown * kb; idx += NT) {
            const int j = idx / kb, t = idx - j * kb;
            Xp[t * SL + j] = __ldcg(X + (size_t)(c + C * j) * N + k0 + t);
            Fo[t * SL + j] = 0.0;
        }
        __syncthreads();
        // ------------------------------------------------------------ panel phase
        for (int s = 0; s < kb; ++s) {
            const int k = k0 + s, par = k & 1;
            // my candidate for column k: largest |x_i[k]| over my slots i >= k (NaN wins: reported as singular)
            double best = -1.0; int bj = -1;
            for (int j = tid; j < nown; j += NT) {
                if (c + C * j < k) continue;
                const double v = fabs(Xp[s * SL + j]);
                if (qmcd_invb_better(v, j, best, bj)) { best = v; bj = j; }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const double ov = __shfl_xor_sync(0xffffffffu, best, o); const int oj = __shfl_xor_sync(0xffffffffu, bj, o);
                if (qmcd_invb_better(ov, oj, best, bj)) { best = ov; bj = oj; }
            }
            if (lane == 0) { s_val[warp] = best; s_idx[warp] = bj; }
            __syncthreads();
            if (tid == 0) {
                double bv = -1.0; int bi = -1;
                for (int w = 0; w < NW; ++w)
                    if (qmcd_invb_better(s_val[w], s_idx[w], bv, bi)) { bv = s_val[w]; bi = s_idx[w]; }
                s_q = bi;
            }
            __syncthreads();
            {
                double* rec = cand + ((size_t)par * C + c) * QMCD_INVB_REC;
                const int jb = s_q;
                if (tid == 0) { rec[0] = (jb >= 0) ? fabs(Xp[s * SL + jb]) : -1.0; rec[1] = (jb >= 0) ? (double)(c + C * jb) : -1.0; }
                if (jb >= 0 && tid < kb) { rec[2 + tid] = Xp[tid * SL + jb]; rec[2 + QMCD_INVB_KB + tid] = Fo[tid * SL + jb]; }
                if (c == k % C && tid < kb) {                  // I own slot k
                    const int jk = (k - c) / C;
                    kdat[(size_t)par * 2 * QMCD_INVB_KB + tid] = Xp[tid * SL + jk];
                    kdat[(size_t)par * 2 * QMCD_INVB_KB + QMCD_INVB_KB + tid] = Fo[tid * SL + jk];
                }
            }
            grid.sync();
            // the walker's pivot slot: largest |.|, lowest slot on ties (the same choice in every CTA)
            if (warp == 0) {
                double bv = -1.0; int bi = -1, bq = -1;
                for (int q = lane; q < C; q += 32) {
                    const double* rec = cand + ((size_t)par * C + q) * QMCD_INVB_REC;
                    const double v = __ldcg(rec); const int i = (int)__ldcg(rec + 1);
                    if (qmcd_invb_better(v, i, bv, bi)) { bv = v; bi = i; bq = q; }
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    const double ov = __shfl_xor_sync(0xffffffffu, bv, o);
                    const int oi = __shfl_xor_sync(0xffffffffu, bi, o), oq = __shfl_xor_sync(0xffffffffu, bq, o);
                    if (qmcd_invb_better(ov, oi, bv, bi)) { bv = ov; bi = oi; bq = oq; }
                }
                if (lane == 0) { s_p = bi; s_q = bq; }
            }
            __syncthreads();
            const int p = (s_p >= 0) ? s_p : k, wq = (s_p >= 0) ? s_q : k % C;
            if (tid < kb) {
                const double* rec = cand + ((size_t)par * C + wq) * QMCD_INVB_REC;
                const double* kd = kdat + (size_t)par * 2 * QMCD_INVB_KB;
                ke[tid] = __ldcg(kd + tid); kf[tid] = __ldcg(kd + QMCD_INVB_KB + tid);
                if (s_p >= 0) { pe[tid] = __ldcg(rec + 2 + tid); pf[tid] = __ldcg(rec + 2 + QMCD_INVB_KB + tid); }
                else { pe[tid] = ke[tid]; pf[tid] = kf[tid]; }
            }
            __syncthreads();
            const double pv = pe[s];
            const bool bad = !(fabs(pv) > 0.0) || !isfinite(pv);
            const double d = bad ? 1.0 : 1.0 / pv;
            if (c == 0 && tid == 0) {
                piv[k] = (s_p >= 0) ? s_p : -1;
                if (bad && a.info[b] == 0) a.info[b] = k + 1;
            }
            if (c == 0 && tid < kb) {                          // row s of L | d | (cleared above the diagonal: filled after the panel)
                lf[s * QMCD_INVB_KB + tid] = (tid < s) ? pf[tid] : (tid == s) ? d : 0.0;
            }
            __syncthreads();
            if (tid < kb) pe[tid] = (tid == s) ? d : pe[tid] * d;     // rho_s on the panel columns
            __syncthreads();
            for (int j = tid; j < nown; j += NT) {
                const int i = c + C * j;
                double* x = Xp + j; double* f = Fo + j;       // entry t at [t * SL]: consecutive slots in consecutive banks
                if (i == k) {
                    for (int t = 0; t < kb; ++t) { x[t * SL] = pe[t]; f[t * SL] = (t == s) ? -1.0 : 0.0; }
                } else {
                    if (i == p) for (int t = 0; t < kb; ++t) { x[t * SL] = ke[t]; f[t * SL] = (t < s) ? kf[t] : 0.0; }
                    const double fs = x[s * SL];
                    x[s * SL] = 0.0;
                    for (int t = 0; t < kb; ++t) x[t * SL] -= fs * pe[t];
                    f[s * SL] = fs;
                }
            }
            // the other columns of rows k and p change places (a column segment per CTA; the panel columns live in shared memory)
            if (p != k) {
                const int seg = (N + C - 1) / C, q0 = c * seg, q1 = min(N, q0 + seg);
                double* xk = X + (size_t)k * N; double* xp = X + (size_t)p * N;
                for (int q = q0 + tid; q < q1; q += NT) {
                    if (q >= k0 && q < k0 + kb) continue;
                    const double u = __ldcg(xk + q), v = __ldcg(xp + q);
                    xk[q] = v; xp[q] = u;
                }
            }
            __syncthreads();
        }
        // ---- panel entries back to the matrix; the pivot slots' later multipliers above the diagonal of lf
        for (int idx = tid; idx < nown * kb; idx += NT) {
            const int j = idx / kb, t = idx - j * kb, i = c + C * j;
            X[(size_t)i * N + k0 + t] = Xp[t * SL + j];
            if (i >= k0 && i < k0 + kb && t > i - k0) lf[(i - k0) * QMCD_INVB_KB + t] = Fo[t * SL + j];
        }
        grid.sync();
        // ------------------------------------------------------------ phase A: my non-pivot slots, the other columns
        auto build_rho = [&](int q0, int cw) {                  // rho[s][q], q < cw, from the pivot rows' chunk (all threads)
            for (int idx = tid; idx < kb * cw; idx += NT) {
                const int s = idx / cw, q = idx - s * cw;
                rho[(size_t)s * CH + q] = __ldcg(X + (size_t)(k0 + s) * N + q0 + q);
            }
            __syncthreads();
            for (int q = tid; q < cw; q += NT)
                for (int s = 0; s < kb; ++s) {
                    double r = rho[(size_t)s * CH + q];
                    for (int t = 0; t < s; ++t) r -= __ldcg(lf + s * QMCD_INVB_KB + t) * rho[(size_t)t * CH + q];
                    rho[(size_t)s * CH + q] = r * __ldcg(lf + s * QMCD_INVB_KB + s);
                }
            __syncthreads();
        };
        for (int q0 = 0; q0 < N; q0 += CH) {
            const int cw = min(CH, N - q0);
            build_rho(q0, cw);
            for (int j = warp; j < nown; j += NW) {
                const int i = c + C * j;
                if (i >= k0 && i < k0 + kb) continue;          // a pivot slot: phase B
                double* xi = X + (size_t)i * N + q0;
                double f[QMCD_INVB_KB];
#pragma unroll
                for (int s = 0; s < QMCD_INVB_KB; ++s) f[s] = (s < kb) ? Fo[s * SL + j] : 0.0;
                if (vec) {                                     // two columns per lane and load, four loads in flight (the pass is bound by bytes in flight)
                    for (int qb = 2 * lane; qb < cw; qb += 256) {
                        double2 x[4], x0[4];
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            const int q = qb + 64 * u;
                            x[u] = (q < cw) ? __ldcg(reinterpret_cast<const double2*>(xi + q)) : make_double2(0.0, 0.0);
                            x0[u] = x[u];
                        }
#pragma unroll
                        for (int s = 0; s < QMCD_INVB_KB; ++s)
                            if (s < kb) {
#pragma unroll
                                for (int u = 0; u < 4; ++u) {
                                    const int q = min(qb + 64 * u, cw - 2);
                                    const double2 r = *reinterpret_cast<const double2*>(rho + (size_t)s * CH + q);
                                    x[u].x -= f[s] * r.x; x[u].y -= f[s] * r.y;
                                }
                            }
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            const int q = qb + 64 * u, qa = q0 + q;
                            if (q >= cw) continue;
                            if (qa >= k0 && qa < k0 + kb) x[u].x = x0[u].x;             // panel columns: already final
                            if (qa + 1 >= k0 && qa + 1 < k0 + kb) x[u].y = x0[u].y;
                            *reinterpret_cast<double2*>(xi + q) = x[u];
                        }
                    }
                } else {
                    for (int q = lane; q < cw; q += 32) {
                        const int qa = q0 + q;
                        if (qa >= k0 && qa < k0 + kb) continue;
                        double x = __ldcg(xi + q);
#pragma unroll
                        for (int s = 0; s < QMCD_INVB_KB; ++s) if (s < kb) x -= f[s] * rho[(size_t)s * CH + q];
                        xi[q] = x;
                    }
                }
            }
            __syncthreads();
        }
        grid.sync();
        // ------------------------------------------------------------ phase B: the pivot slots, chunks dealt over my walker's CTAs
        for (int q0 = c * CH; q0 < N; q0 += C * CH) {
            const int cw = min(CH, N - q0);
            build_rho(q0, cw);
            for (int idx = tid; idx < kb * cw; idx += NT) {
                const int s = idx / cw, q = idx - s * cw, qa = q0 + q;
                if (qa >= k0 && qa < k0 + kb) continue;
                double r = rho[(size_t)s * CH + q];
                for (int t = s + 1; t < kb; ++t) r -= __ldcg(lf + s * QMCD_INVB_KB + t) * rho[(size_t)t * CH + q];
                X[(size_t)(k0 + s) * N + qa] = r;
            }
            __syncthreads();
        }
        grid.sync();
    }
    // ---- undo the row swaps as column swaps, last first, composed into one gather per row
    double* rowp = reinterpret_cast<double*>(invb_smem);
    int* cols = reinterpret_cast<int*>(rowp + N);
    __syncthreads();
    if (tid == 0) {
        for (int q = 0; q < N; ++q) cols[q] = q;
        for (int k = N - 1; k >= 0; --k) {
            const int p = __ldcg(piv + k);
            if (p >= 0 && p != k) { const int t = cols[k]; cols[k] = cols[p]; cols[p] = t; }
        }
    }
    __syncthreads();
    for (int i = c; i < N; i += C) {
        double* xi = X + (size_t)i * N;
        for (int q = tid; q < N; q += NT) rowp[q] = __ldcg(xi + q);
        __syncthreads();
        for (int q = tid; q < N; q += NT) xi[q] = rowp[cols[q]];
        __syncthreads();
    }
}
