// qmcd_invert.cuh -- batched on-device inversion of the Slater matrices:
// the "explicit copy of the matrix inverse" of PAPER.md:63 that qmcd_set_inverse adopts, and
// the periodic fresh inversion that bounds the rounding drift of the updates.
//
// In-place Gauss-Jordan elimination with partial (row) pivoting, one cooperative launch for
// the whole batch: walker b is owned by C CTAs, CTA c holding the row slots i == c (mod C).
// Step k (two grid barriers):
//   1. every CTA has published its candidate max |X[i][k]|, i >= k (found while it wrote those
//      values in step k-1); after the barrier all CTAs of the walker pick the same pivot slot p
//      and stage OLD rows p (pivot) and k into shared memory;
//   2. after the second barrier (nobody still reads rows p / k from global memory) every CTA
//      rewrites its slots:  slot k <- pivot row / pivot (pivot column entry := 1/pivot),
//      slot p <- old row k eliminated, any other slot i <- row i eliminated
//      (eliminated: f = x[k]; x[k] := 0; x -= f * new row k).
// The row swaps are undone at the end as column swaps in reverse order (composed into one
// gather per row).  HBM-bound by construction (every step streams the matrix once: 16 N^3
// bytes per walker); a blocked, DMMA-fed variant is round-2 work -- this is a set-up step,
// not part of the timed hot path.
#pragma once
#include <cuda_runtime.h>
#include <cooperative_groups.h>
#include <stdint.h>

#define QMCD_INV_THREADS 512      // largest CTA; the host launches 256 or 512 threads, whichever puts more warps on an SM
#define QMCD_INV_CMAX 256       // candidate slots per walker in the scratch area

struct QmcdInvArgs {
    int N, batch, C;
    const double* A;            // [batch][N][N] row-major
    double* X;                  // [batch][N][N] result (may alias A)
    int* piv;                   // [batch][N]    pivot slot of every step
    double* cand_val;           // [batch][CMAX]
    int* cand_idx;              // [batch][CMAX]
    int* info;                  // [batch] 0, or k+1 of the first zero / non-finite pivot
};

__global__ void __launch_bounds__(QMCD_INV_THREADS, 2) qmcd_invert_kernel(const QmcdInvArgs a) {
    namespace cg = cooperative_groups;
    extern __shared__ __align__(16) unsigned char inv_smem[];
    cg::grid_group grid = cg::this_grid();
    const int N = a.N, C = a.C;
    const int b = blockIdx.x / C, c = blockIdx.x - b * C;
    const int NT = (int)blockDim.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, NW = NT >> 5;
    double* rowp = reinterpret_cast<double*>(inv_smem);     // [N] new row k (scaled pivot row)
    double* rowk = rowp + N;                                // [N] old row k
    int* cols = reinterpret_cast<int*>(rowk) + N;           // [N] final column gather (rowk is dead by then: piv | cols)
    __shared__ double s_val[QMCD_INV_THREADS / 32];
    __shared__ int s_idx[QMCD_INV_THREADS / 32];
    __shared__ int s_p;
    const double* Ab = a.A + (size_t)b * N * N;
    double* X = a.X + (size_t)b * N * N;
    double* cval = a.cand_val + (size_t)b * QMCD_INV_CMAX;
    int* cidx = a.cand_idx + (size_t)b * QMCD_INV_CMAX;
    int* piv = a.piv + (size_t)b * N;
    const bool vec = ((N & 1) == 0) && ((reinterpret_cast<uintptr_t>(X) & 15) == 0);

    // copy my rows, candidates for column 0
    double best = -1.0; int besti = -1;
    for (int i = c + C * warp; i < N; i += C * NW) {
        for (int k = lane; k < N; k += 32) X[(size_t)i * N + k] = Ab[(size_t)i * N + k];
        const double v = fabs(Ab[(size_t)i * N]);
        if (!(v <= best)) { best = v; besti = i; }           // NaN wins: reported as singular below
    }
    for (int k = 0; k < N; ++k) {
        // ---- publish this CTA's candidate for column k
        if (lane == 0) { s_val[warp] = best; s_idx[warp] = besti; }
        __syncthreads();
        if (tid == 0) {
            double bv = -1.0; int bi = -1;
            for (int w = 0; w < NW; ++w)
                if (s_idx[w] >= 0 && (!(s_val[w] <= bv) || (s_val[w] == bv && s_idx[w] < bi))) { bv = s_val[w]; bi = s_idx[w]; }
            cval[c] = bv; cidx[c] = bi;
        }
        grid.sync();
        // ---- the walker's pivot slot (same choice in every CTA: largest |.|, lowest slot on ties)
        if (tid == 0) {
            double bv = -1.0; int bi = -1;
            for (int q = 0; q < C; ++q) {
                const double v = __ldcg(cval + q); const int i = __ldcg(cidx + q);
                if (i >= 0 && (!(v <= bv) || (v == bv && i < bi))) { bv = v; bi = i; }
            }
            s_p = bi;
            if (c == 0) piv[k] = bi;
        }
        __syncthreads();
        const int p = (s_p >= 0) ? s_p : k;
        for (int q = tid; q < N; q += NT) {
            rowp[q] = __ldcg(X + (size_t)p * N + q);
            rowk[q] = __ldcg(X + (size_t)k * N + q);
        }
        __syncthreads();
        const double pv = rowp[k];
        const bool bad = !(fabs(pv) > 0.0) || !isfinite(pv);
        if (bad && c == 0 && tid == 0 && a.info[b] == 0) a.info[b] = k + 1;
        const double d = bad ? 1.0 : 1.0 / pv;
        __syncthreads();
        for (int q = tid; q < N; q += NT) rowp[q] = (q == k) ? d : rowp[q] * d;
        grid.sync();                                         // every CTA holds rows p and k: slots may change
        // ---- rewrite my slots; collect candidates for column k+1 on the way
        best = -1.0; besti = -1;
        const int kn = k + 1;
        for (int i = c + C * warp; i < N; i += C * NW) {
            double* xi = X + (size_t)i * N;
            if (i == k) {
                for (int q = lane; q < N; q += 32) xi[q] = rowp[q];
                continue;
            }
            const bool from_k = (i == p);                    // slot p receives old row k (the swap)
            const double f = from_k ? rowk[k] : __ldcg(xi + k);
            double cand = 0.0;
            int src_lane;
            if (vec) {                                       // 16-byte accesses, four rows of loads in flight per lane
                const double2* rp2 = reinterpret_cast<const double2*>(rowp);
                const double2* rk2 = reinterpret_cast<const double2*>(rowk);
                double2* x2 = reinterpret_cast<double2*>(xi);
                const int N2 = N >> 1, k2 = k >> 1, kn2 = kn >> 1;
#pragma unroll 4
                for (int q = lane; q < N2; q += 32) {
                    const double2 x = from_k ? rk2[q] : __ldcg(x2 + q);
                    const double2 rr = rp2[q];
                    double2 y;
                    y.x = x.x - f * rr.x; y.y = x.y - f * rr.y;
                    if (q == k2) { if (k & 1) y.y = -f * rr.y; else y.x = -f * rr.x; }
                    x2[q] = y;
                    if (q == kn2) cand = (kn & 1) ? y.y : y.x;
                }
                src_lane = kn2 & 31;
            } else {
                for (int q = lane; q < N; q += 32) {
                    const double x = from_k ? rowk[q] : __ldcg(xi + q);
                    const double y = (q == k) ? -f * rowp[q] : x - f * rowp[q];
                    xi[q] = y;
                    if (q == kn) cand = y;
                }
                src_lane = kn & 31;
            }
            if (kn < N && i > k) {
                cand = fabs(__shfl_sync(0xffffffffu, cand, src_lane));
                if (!(cand <= best)) { best = cand; besti = i; }
            }
        }
        __syncthreads();                                     // rowp / rowk / s_p are restaged next step
    }
    grid.sync();
    // ---- undo the row swaps as column swaps, last first, composed into one gather per row
    int* piv_s = reinterpret_cast<int*>(rowk);
    for (int q = tid; q < N; q += NT) piv_s[q] = __ldcg(piv + q);
    __syncthreads();
    if (tid == 0) {
        for (int q = 0; q < N; ++q) cols[q] = q;
        for (int k = N - 1; k >= 0; --k) {
            const int p = piv_s[k];
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
