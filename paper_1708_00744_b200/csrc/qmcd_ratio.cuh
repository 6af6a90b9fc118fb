// qmcd_ratio.cuh -- F1 for the per-call API (qmcd_ratio / qmcd_ratio_jv): the look-ahead determinant ratio of
// Eqs. 1 and 3 as a bandwidth kernel of its own,
//     d = B0[j,:].v ;  p_i = B0[j,:].C[i,:] - delta(j, j_i) ;  q_i = W[i,:].v  (i < m) ;  R = d - p^T M q.
// A walker's 2m + 2 length-N streams are cut into G column slices x GR groups of queue rows: one small CTA
// (256 threads, <= 64 registers, a few KB of shared memory, several CTAs per SM) per (slice, row group, walker).
// A warp takes queue rows; every lane issues all its 16-byte loads of a row pair before the first FMA, reduces
// with shuffles and stores the partial sums.  The last CTA of a walker to finish (atomic ticket) adds the
// partials in slice order -- so the result does not depend on which CTA that was --, finishes the m x m part
// (c = M q, r = M^T p with M from global memory) and stages R, c, r for qmcd_accept.  The slices of v and
// B0[j,:] are also written to slot m of C and W, the slot the move takes if accepted.
#pragma once
#include "qmcd_dev.cuh"

struct QmcdRatioArgs {
    QmcdDev P;
    int j;                    // electron (all walkers) when jv == nullptr
    const int* jv;            // [batch] per-walker electron or nullptr
    const double* v;          // [batch][N]
    double* R_out;            // [batch]
    double* part;             // [batch][G][2K + 2] partial sums
    unsigned* cnt;            // [batch] tickets (self-resetting)
    int G, GR;                // column slices, row groups
    int slice;                // columns per slice (multiple of VEC)
};

#define QMCD_RATIO_NU 4       // most vectors per lane and row: slice <= 128 * VEC columns
#define QMCD_RATIO_RB 2       // queue-row pairs whose loads a warp issues together

template <int VEC> struct QmcdVec;
template <> struct QmcdVec<2> {
    typedef double2 T;
    static __device__ __forceinline__ T ld(const double* p) { T v; asm volatile("ld.global.cg.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p)); return v; }
    static __device__ __forceinline__ void st(double* p, T v) { *reinterpret_cast<double2*>(p) = v; }
    static __device__ __forceinline__ T zero() { return make_double2(0.0, 0.0); }
    static __device__ __forceinline__ double dot(T a, T b, double acc) { return fma(a.y, b.y, fma(a.x, b.x, acc)); }
};
template <> struct QmcdVec<1> {
    typedef double T;
    static __device__ __forceinline__ T ld(const double* p) { return __ldcg(p); }
    static __device__ __forceinline__ void st(double* p, T v) { *p = v; }
    static __device__ __forceinline__ T zero() { return 0.0; }
    static __device__ __forceinline__ double dot(T a, T b, double acc) { return fma(a, b, acc); }
};

// NU = vectors per lane and row (slice = 32 NU VEC columns).  The host sizes the grid to ONE wave of resident CTAs
// (a second, short wave costs a full ramp of dependent memory round trips on a kernel that lasts ~15 us).
template <int VEC, int NU>
__global__ void __launch_bounds__(QMCD_THREADS, (NU <= 2) ? 4 : 3) qmcd_ratio_kernel(const QmcdRatioArgs A) {
    typedef QmcdVec<VEC> V;
    extern __shared__ __align__(16) double rsm[];             // last CTA only: pf | qf | cf | rf, K doubles each
    __shared__ int s_last;
    const QmcdDev& P = A.P;
    const int N = P.N, K = P.K;
    const int b = blockIdx.z, gc = blockIdx.x, gr = blockIdx.y;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int m = __ldcg(P.m + b);
    const int j = A.jv ? A.jv[b] : A.j;
    if (j < 0 || j >= N) {                                    // uniform over the walker's CTAs: nobody takes a ticket
        if (gc == 0 && gr == 0 && tid == 0) { qmcd_set_status(P, QMCD_DEV_EINVAL, b, P.counters[(size_t)b * 8]); P.sj[b] = -1; A.R_out[b] = 0.0; }
        return;
    }
    const int lo = gc * A.slice, hi = min(N, lo + A.slice);
    const double* rowj = P.B + ((size_t)b * N + j) * N;
    const double* vv = A.v + (size_t)b * N;
    const double* Cw = P.C + (size_t)b * K * N;
    const double* Ww = P.W + (size_t)b * K * N;
    double* pp = A.part + ((size_t)b * A.G + gc) * (2 * K + 2);

    // this lane's elements of the slice: k = lo + VEC (lane + 32 u)
    typename V::T rj[NU], vx[NU];
#pragma unroll
    for (int u = 0; u < NU; ++u) {
        const int k = lo + VEC * (lane + 32 * u);
        rj[u] = (k < hi) ? V::ld(rowj + k) : V::zero();
        vx[u] = (k < hi) ? V::ld(vv + k) : V::zero();
    }
    if (gr == 0 && wid == 0) {
        double d = 0.0;
#pragma unroll
        for (int u = 0; u < NU; ++u) d = V::dot(rj[u], vx[u], d);
        d = qmcd_warp_sum(d);
        if (lane == 0) pp[2 * K] = d;
        // stage the move's slot: W[m] <- B0[j,:], C[m] <- v (this slice)
        if (m < K) {
            double* Wm = P.W + ((size_t)b * K + m) * N;
            double* Cm = P.C + ((size_t)b * K + m) * N;
#pragma unroll
            for (int u = 0; u < NU; ++u) {
                const int k = lo + VEC * (lane + 32 * u);
                if (k < hi) { V::st(Wm + k, rj[u]); V::st(Cm + k, vx[u]); }
            }
        }
    }
    // queue rows i = 8 gr + wid, step 8 GR, QMCD_RATIO_RB of them at a time: all loads of the row pairs (C[i], W[i]) are issued
    // before the first FMA
    const int istep = QMCD_WARPS * A.GR;
    for (int i0 = gr * QMCD_WARPS + wid; i0 < m; i0 += istep * QMCD_RATIO_RB) {
        typename V::T cv[QMCD_RATIO_RB][NU], wv[QMCD_RATIO_RB][NU];
#pragma unroll
        for (int r = 0; r < QMCD_RATIO_RB; ++r) {
            const int i = i0 + r * istep;
            const double* Ci = Cw + (size_t)i * N;
            const double* Wi = Ww + (size_t)i * N;
#pragma unroll
            for (int u = 0; u < NU; ++u) {
                const int k = lo + VEC * (lane + 32 * u);
                const bool ok = (i < m) && (k < hi);
                cv[r][u] = ok ? V::ld(Ci + k) : V::zero();
                wv[r][u] = ok ? V::ld(Wi + k) : V::zero();
            }
        }
#pragma unroll
        for (int r = 0; r < QMCD_RATIO_RB; ++r) {
            const int i = i0 + r * istep;
            double p = 0.0, q = 0.0;
#pragma unroll
            for (int u = 0; u < NU; ++u) { p = V::dot(rj[u], cv[r][u], p); q = V::dot(wv[r][u], vx[u], q); }
            p = qmcd_warp_sum(p); q = qmcd_warp_sum(q);
            if (lane == 0 && i < m) { pp[i] = p; pp[K + i] = q; }
        }
    }
    // ---- ticket: the last CTA of this walker finishes the job
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        const unsigned total = (unsigned)(A.G * A.GR);
        const unsigned old = atomicAdd(A.cnt + b, 1u);
        s_last = (old == total - 1);
        if (s_last) A.cnt[b] = 0;                             // ready for the next call (stream order)
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double *pf = rsm, *qf = rsm + K, *cf = rsm + 2 * K, *rf = rsm + 3 * K;
    const double* pb = A.part + (size_t)b * A.G * (2 * K + 2);
    const int* Jw = P.J + (size_t)b * K;
    for (int i = tid; i < m; i += QMCD_THREADS) {
        double p = 0.0, q = 0.0;
        for (int g = 0; g < A.G; ++g) { p += __ldcg(pb + (size_t)g * (2 * K + 2) + i); q += __ldcg(pb + (size_t)g * (2 * K + 2) + K + i); }
        if (__ldcg(Jw + i) == j) p -= 1.0;
        pf[i] = p; qf[i] = q;
    }
    double d = 0.0;
    for (int g = 0; g < A.G; ++g) d += __ldcg(pb + (size_t)g * (2 * K + 2) + 2 * K);
    __syncthreads();
    // c = M q and r = M^T p: 8 threads per index, M (m x m, row stride ldMg) from global memory
    {
        const double* Mb = P.M + (size_t)b * P.ldMg * P.ldMg;
        const int ld = P.ldMg, h = tid & 7;
        for (int x0 = 0; x0 < m; x0 += QMCD_THREADS / 8) {
            const int x = x0 + (tid >> 3);
            double ca = 0.0, ra = 0.0;
            if (x < m)
                for (int y = h; y < m; y += 8) {
                    ca += __ldcg(Mb + (size_t)x * ld + y) * qf[y];
                    ra += pf[y] * __ldcg(Mb + (size_t)y * ld + x);
                }
#pragma unroll
            for (int o = 4; o > 0; o >>= 1) { ca += __shfl_xor_sync(0xffffffffu, ca, o); ra += __shfl_xor_sync(0xffffffffu, ra, o); }
            if (x < m && h == 0) { cf[x] = ca; rf[x] = ra; }
        }
    }
    __syncthreads();
    if (wid == 0) {
        double acc = 0.0;
        for (int a = lane; a < m; a += 32) acc += pf[a] * cf[a];
        acc = qmcd_warp_sum(acc);
        if (lane == 0) { const double R = d - acc; P.sR[b] = R; P.sj[b] = j; A.R_out[b] = R; }
    }
    for (int i = tid; i < m; i += QMCD_THREADS) { P.sc[(size_t)b * K + i] = cf[i]; P.sr[(size_t)b * K + i] = rf[i]; }
}
