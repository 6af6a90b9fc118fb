// qmcd_flush_tma.cuh -- the rank-m flush of Eq. 4 for K <= 64, one tile of 128 rows
// of B per call, with every operand brought into shared memory by TMA (cp.async.bulk.tensor + mbarrier)
// and the eight warps doing nothing but LDS + DMMA.8x8x4 in straight-line code:
//
//     iterations 0 .. nk-1      (nk = N/32)   T  = B0[tile, 32 k-columns] . C[:, same]^T   accumulated in registers
//     iteration  nk                            T  = -T + E_J ;  T <- T M                   (M = S^-1, 64 x 64, zero outside m x m)
//     iterations nk+1 .. 2nk                   B[tile, 32 columns] += T . W[:, same]       written back from registers
//
// T NEVER LEAVES THE REGISTERS: with the permuted contraction index of qmcd_flush_mma.cuh (k-slot c of k-step s
// is k = 8q + 2c + s) the accumulator fragment of n-tile q -- lane (g, c) holds T[g][8q + 2c], T[g][8q + 2c + 1] --
// IS the A fragment of k-group q of the next product.  A warp owns 16 rows of the tile through all three parts.
//
// One ring of 4 stages of 48 KB carries everything else; stage contents per kind of iteration:
//     NT : B0 tile as [4 k-groups][128 rows][8]      + C as [4 k-groups][8 NB rows][8]          (4-D tensor maps, no swizzle:
//          an 8 x 8 fp64 fragment block is 512 contiguous bytes, so the 16-byte fragment loads are conflict-free)
//     M  : M as [4 column groups][64 rows][16]       (SWIZZLE_128B: 16-byte chunk ^= row % 8; read with 8-byte loads,
//          n-slot g of tile t = column 8t + g, conflict-free under the same k permutation)
//     NN : B0 tile as [4 column groups][128 rows][8] + W as [2 column groups][8 NB rows][16]   (W swizzled like M, read
//          with 16-byte loads: n-slot g of tile t of group G is column 16G + 2g + t)
// Lane 0 of warp (j mod 8) issues, at the top of iteration j, the loads of iteration j + 3 into the stage every warp
// left in iteration j - 1.  Rows past N and queue rows past K are zero-filled by TMA.  Any rank m <= K runs the
// full 8 NB columns: M is zero outside m x m, so the stale (finite) queue rows past m contribute exact zeros.
#pragma once
#include <cuda.h>
#include "qmcd_flush_mma.cuh"

// 4-D views, see qmcd_api.cu.  B, B64, C, W, M, Y: the flush (this file; B64: 64-row boxes of B; Y = M W (K > 64), viewed
// like W).  Bs, Vs, C32, W32: the look-ahead ring of qmcd_superblock.cuh -- boxes of 2 k-groups (k-major view): 16 / 32 / 64
// rows of B, as many proposals of the current qmcd_sweep launch, 32 rows of C and of W.
struct QmcdTmaps { CUtensorMap B, C, W, M, B64, Y, C32, W32, Bs[3], Vs[3]; };

#define QMCD_TMA_NS 4
#define QMCD_TMA_STAGE_BYTES 49152
#define QMCD_TMA_BAR_OFF 512                 // full[NS], empty[NS] mbarriers inside the shared-memory header
#define QMCD_TMA_STAGE_OFF 1024              // stages are 1024-byte aligned (swizzle atoms)
#define QMCD_TMA_ROWS 128
__host__ __device__ inline size_t qmcd_flush_tma_smem_bytes() {
    return (size_t)QMCD_TMA_STAGE_OFF + QMCD_TMA_NS * QMCD_TMA_STAGE_BYTES;
}
__host__ __device__ inline int qmcd_tma_NB(int K) { return K <= 8 ? 1 : K <= 16 ? 2 : K <= 32 ? 4 : K <= 64 ? 8 : 16; }

__device__ __forceinline__ unsigned qmcd_su32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void qmcd_mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void qmcd_mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void qmcd_mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void qmcd_mbar_wait(unsigned bar, unsigned parity) {
    asm volatile("{\n\t.reg .pred P1;\n\tLAB_WAIT:\n\tmbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t@P1 bra DONE;\n\tbra LAB_WAIT;\n\tDONE:\n\t}"
                 :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void qmcd_tma_load4(unsigned dst, const CUtensorMap* tm, int c0, int c1, int c2, int c3, unsigned bar) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 :: "r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar) : "memory");
}
// 1-D bulk copies (rows of the queue append): global -> shared with mbarrier completion, shared -> global as a bulk group
__device__ __forceinline__ void qmcd_bulk_load(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void qmcd_bulk_store(void* dst, unsigned src, unsigned bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" :: "l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void qmcd_bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void qmcd_bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void qmcd_bulk_wait_read1() { asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory"); }
__device__ __forceinline__ void qmcd_bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
// L2 eviction policies: the flush streams each tile of B once per pass (evict first: do not push the queues
// out of L2); the queue rows C, W and M are re-read by every tile and every look-ahead block (evict last)
__device__ __forceinline__ unsigned long long qmcd_policy_evict_first() {
    unsigned long long p; asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p)); return p;
}
__device__ __forceinline__ unsigned long long qmcd_policy_evict_last() {
    unsigned long long p; asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p)); return p;
}
__device__ __forceinline__ void qmcd_tma_load4_hint(unsigned dst, const CUtensorMap* tm, int c0, int c1, int c2, int c3, unsigned bar,
                                                    unsigned long long policy) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4, %5}], [%6], %7;"
                 :: "r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar), "l"(policy) : "memory");
}
__device__ __forceinline__ void qmcd_fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

// look-ahead ring (qmcd_superblock.cuh): 3 stages; full[3] at +576, empty[3] at +600 (the append's barriers: +640 ... +768)
#define QMCD_LA_NS 3
#define QMCD_LA_BAR_OFF 576
__device__ __forceinline__ void qmcd_la_init_barriers(unsigned char* smem) {
    const unsigned bar0 = qmcd_su32(smem + QMCD_LA_BAR_OFF);
#pragma unroll
    for (int s = 0; s < QMCD_LA_NS; ++s) {
        qmcd_mbar_init(bar0 + 8 * s, 1);
        qmcd_mbar_init(bar0 + 8 * QMCD_LA_NS + 8 * s, QMCD_WARPS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

// once per kernel, by one thread, before the CTA's first barrier
__device__ __forceinline__ void qmcd_tma_init_barriers(unsigned char* smem) {
    const unsigned bar0 = qmcd_su32(smem + QMCD_TMA_BAR_OFF);
#pragma unroll
    for (int s = 0; s < QMCD_TMA_NS; ++s) {
        qmcd_mbar_init(bar0 + 8 * s, 1);                                   // full: the issuing thread's expect_tx arrival
        qmcd_mbar_init(bar0 + 8 * QMCD_TMA_NS + 8 * s, QMCD_WARPS);        // empty: one arrival per warp
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

// One tile of 64 A_T rows.  `itc` = iterations this CTA has pushed through the ring so far (the same in every
// thread; it fixes stage and mbarrier parity), updated on return.  All 256 threads; ends without a CTA barrier.
//   YP = false (K <= 64): the three parts above, M applied in registers.
//   YP = true  (64 < K <= 128, NB = 16, A_T = 1): Y = M W was formed by the job's first phase; part 2 is only
//              T = -T + E_J and part 3 multiplies by Y (tensor map TM.Y) -- 2 nk iterations, no M stage.
template <int NB, int A_T, bool YP>
__device__ __noinline__ void qmcd_flush_tile_tma(const QmcdDev& P, const QmcdTmaps& TM, unsigned char* smem, int b, int m, int tile,
                                                 unsigned& itc) {
    constexpr int ROWS = 64 * A_T;
    constexpr unsigned OFF2 = 256u * ROWS;                     // second operand of a stage, after the B tile
    constexpr unsigned TX_ROWS = OFF2 + 2048u * NB;
    constexpr int NS = QMCD_TMA_NS;
    constexpr bool DB = (NB <= 8);                             // double-buffered fragments while the registers allow
    static_assert(OFF2 + 2048u * NB <= QMCD_TMA_STAGE_BYTES, "stage too small");
    const int N = P.N, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, g = lane >> 2, c = lane & 3;
    const int nk = N / 32, total = YP ? 2 * nk : 2 * nk + 1, nn0 = YP ? nk : nk + 1;
    const int row0 = tile * ROWS, wrow = wid * 8 * A_T;
    const unsigned bar0 = qmcd_su32(smem + QMCD_TMA_BAR_OFF);
    unsigned char* st0 = smem + QMCD_TMA_STAGE_OFF;
    const unsigned it0 = itc;
    double* Bw = P.B + (size_t)b * N * N;
    const CUtensorMap* tmB = (A_T == 2) ? &TM.B : &TM.B64;

    const unsigned long long pol_stream = qmcd_policy_evict_first(), pol_keep = qmcd_policy_evict_last();
    // (measured: loading part 1's tile without the evict-first hint when all tiles in flight fit in L2 -- 64-row tiles on c2,
    // 74 MB -- does not turn part 3's second read into L2 hits: c2 K = 16 3.10 vs 3.20 M moves/s)
    auto issue = [&](int j) {                     // one thread: the loads of iteration j of this tile
        const unsigned gi = it0 + (unsigned)j, s = gi % NS, u = gi / NS;
        if (u > 0) qmcd_mbar_wait(bar0 + 8 * NS + 8 * s, (u - 1) & 1);               // every warp has left the stage
        const unsigned dst = qmcd_su32(st0 + s * QMCD_TMA_STAGE_BYTES), fb = bar0 + 8 * s;
        if (j < nk) {
            qmcd_mbar_expect_tx(fb, TX_ROWS);
            qmcd_tma_load4_hint(dst, tmB, 0, row0, 4 * j, b, fb, pol_stream);
            qmcd_tma_load4_hint(dst + OFF2, &TM.C, 0, 0, 4 * j, b, fb, pol_keep);
        } else if (!YP && j == nk) {
            qmcd_mbar_expect_tx(fb, 32768u);
            qmcd_tma_load4_hint(dst, &TM.M, 0, 0, 0, b, fb, pol_keep);
        } else {
            const int jj = j - nn0;
            qmcd_mbar_expect_tx(fb, TX_ROWS);
            qmcd_tma_load4_hint(dst, tmB, 0, row0, 4 * jj, b, fb, pol_stream);
            qmcd_tma_load4_hint(dst + OFF2, YP ? &TM.Y : &TM.W, 0, 0, 2 * jj, b, fb, pol_keep);
        }
    };
    if (tid == 0) {
#pragma unroll
        for (int j = 0; j < NS - 1; ++j) issue(j);            // total >= 2 * 4 > NS - 1
    }

    // T for this warp's 8 A_T rows: T[a][q][e] = T[row wrow + 8 a + g][column 8 q + 2 c + e]
    double T[A_T][NB][2];
#pragma unroll
    for (int a = 0; a < A_T; ++a)
#pragma unroll
        for (int q = 0; q < NB; ++q) { T[a][q][0] = 0.0; T[a][q][1] = 0.0; }

    // ---------------- NT: T = B0[tile,:] C^T, 4 k-groups of 8 columns per iteration
    for (int j = 0; j < nk; ++j) {
        const unsigned gi = it0 + (unsigned)j, s = gi % NS, u = gi / NS;
        const unsigned char* stg = st0 + s * QMCD_TMA_STAGE_BYTES;
        qmcd_mbar_wait(bar0 + 8 * s, u & 1);
        if (wid == (j & 7) && lane == 0 && j + NS - 1 < total) issue(j + NS - 1);
        const unsigned As = qmcd_su32(stg) + 8u * ((wrow + g) * 8 + 2 * c);        // byte addresses in shared memory
        const unsigned Cs = qmcd_su32(stg) + OFF2 + 8u * (g * 8 + 2 * c);
        if (DB) {
            double2 av[2][A_T], bv[2][NB];
#pragma unroll
            for (int a = 0; a < A_T; ++a) av[0][a] = qmcd_lds128s(As + a * 512);
#pragma unroll
            for (int bt = 0; bt < NB; ++bt) bv[0][bt] = qmcd_lds128s(Cs + bt * 512);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int cur = q & 1, nxt = cur ^ 1;
                if (q < 3) {
#pragma unroll
                    for (int a = 0; a < A_T; ++a) av[nxt][a] = qmcd_lds128s(As + (q + 1) * (ROWS * 64) + a * 512);
#pragma unroll
                    for (int bt = 0; bt < NB; ++bt) bv[nxt][bt] = qmcd_lds128s(Cs + (q + 1) * (512 * NB) + bt * 512);
                }
#pragma unroll
                for (int bt = 0; bt < NB; ++bt)
#pragma unroll
                    for (int a = 0; a < A_T; ++a) qmcd_dmma(T[a][bt][0], T[a][bt][1], av[cur][a].x, bv[cur][bt].x);
#pragma unroll
                for (int bt = 0; bt < NB; ++bt)
#pragma unroll
                    for (int a = 0; a < A_T; ++a) qmcd_dmma(T[a][bt][0], T[a][bt][1], av[cur][a].y, bv[cur][bt].y);
            }
        } else {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                double2 av[A_T];
#pragma unroll
                for (int a = 0; a < A_T; ++a) av[a] = qmcd_lds128s(As + q * (ROWS * 64) + a * 512);
#pragma unroll
                for (int h = 0; h < NB; h += 8) {          // 8 n-tiles at a time: 8 fragment registers pairs live
                    double2 bv[8];
#pragma unroll
                    for (int bt = 0; bt < 8; ++bt) bv[bt] = qmcd_lds128s(Cs + q * (512 * NB) + (h + bt) * 512);
#pragma unroll
                    for (int bt = 0; bt < 8; ++bt)
#pragma unroll
                        for (int a = 0; a < A_T; ++a) qmcd_dmma(T[a][h + bt][0], T[a][h + bt][1], av[a].x, bv[bt].x);
#pragma unroll
                    for (int bt = 0; bt < 8; ++bt)
#pragma unroll
                        for (int a = 0; a < A_T; ++a) qmcd_dmma(T[a][h + bt][0], T[a][h + bt][1], av[a].y, bv[bt].y);
                }
            }
        }
        __syncwarp();
        if (lane == 0) qmcd_mbar_arrive(bar0 + 8 * NS + 8 * s);                      // this warp has left stage s
    }

    // ---------------- T = -T + E_J  (and, K <= 64, T <- T M: iteration nk, the stage holds M)
    {
        const int* Jw = P.J + (size_t)b * P.K;
#pragma unroll
        for (int q = 0; q < NB; ++q)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int i = 8 * q + 2 * c + e;
                const int jr = (i < m) ? __ldcg(Jw + i) - row0 - wrow - g : -1;          // E_J[j_i, i] = 1
#pragma unroll
                for (int a = 0; a < A_T; ++a)
                    T[a][q][e] = (YP && i >= m) ? 0.0 : ((jr == 8 * a) ? 1.0 : 0.0) - T[a][q][e];   // (YP: rows >= m of Y are stale)
            }
    }
    if (!YP) {
        const int j = nk;
        const unsigned gi = it0 + (unsigned)j, s = gi % NS, u = gi / NS;
        const unsigned char* stg = st0 + s * QMCD_TMA_STAGE_BYTES;
        qmcd_mbar_wait(bar0 + 8 * s, u & 1);
        if (wid == (j & 7) && lane == 0 && j + NS - 1 < total) issue(j + NS - 1);
        double T2[A_T][NB][2];
#pragma unroll
        for (int a = 0; a < A_T; ++a)
#pragma unroll
            for (int t = 0; t < NB; ++t) { T2[a][t][0] = 0.0; T2[a][t][1] = 0.0; }
        // M[k][n] at group (n / 16): row k, 16-byte chunk ((n % 16) / 2) ^ (k % 8), half n % 2;  k = 8q + 2c + s, n = 8t + g
        const unsigned Ms = qmcd_su32(stg) + (2 * c) * 128 + (g & 1) * 8;
        const int ch0 = (g >> 1) ^ (2 * c), ch1 = (g >> 1) ^ (2 * c + 1);            // chunk of n-tile parity 0; parity 1: ^ 4
#pragma unroll
        for (int q = 0; q < NB; ++q) {
            double b0[NB], b1[NB];
#pragma unroll
            for (int t = 0; t < NB; ++t) {
                const unsigned pm = Ms + (t >> 1) * 8192 + q * 1024;
                b0[t] = qmcd_lds64s(pm + ((ch0 ^ ((t & 1) << 2)) << 4));
                b1[t] = qmcd_lds64s(pm + 128 + ((ch1 ^ ((t & 1) << 2)) << 4));
            }
#pragma unroll
            for (int t = 0; t < NB; ++t)
#pragma unroll
                for (int a = 0; a < A_T; ++a) qmcd_dmma(T2[a][t][0], T2[a][t][1], T[a][q][0], b0[t]);
#pragma unroll
            for (int t = 0; t < NB; ++t)
#pragma unroll
                for (int a = 0; a < A_T; ++a) qmcd_dmma(T2[a][t][0], T2[a][t][1], T[a][q][1], b1[t]);
        }
#pragma unroll
        for (int a = 0; a < A_T; ++a)
#pragma unroll
            for (int t = 0; t < NB; ++t) { T[a][t][0] = T2[a][t][0]; T[a][t][1] = T2[a][t][1]; }
        __syncwarp();
        if (lane == 0) qmcd_mbar_arrive(bar0 + 8 * NS + 8 * s);
    }

    // ---------------- NN: B[tile, 32 columns] += T X[:, same] (X = W, or Y when YP); initial values from the staged
    // tile, results by STG
    const int sw0 = (g ^ (2 * c)) << 4, sw1 = (g ^ (2 * c + 1)) << 4;
    for (int j = nn0; j < total; ++j) {
        const unsigned gi = it0 + (unsigned)j, s = gi % NS, u = gi / NS;
        const unsigned char* stg = st0 + s * QMCD_TMA_STAGE_BYTES;
        const int n0 = 32 * (j - nn0);
        qmcd_mbar_wait(bar0 + 8 * s, u & 1);
        if (wid == (j & 7) && lane == 0 && j + NS - 1 < total) issue(j + NS - 1);
        const unsigned Ds = qmcd_su32(stg);                                           // [4 groups of 8 columns][ROWS][8]
        const unsigned Ws = Ds + OFF2 + (2 * c) * 128;                                // [2 groups of 16 columns][8 NB rows][128 B]
        double an[A_T][2][2][2];                                                     // [a][G][t][e]
#pragma unroll
        for (int a = 0; a < A_T; ++a)
#pragma unroll
            for (int G = 0; G < 2; ++G) {              // this lane's columns 16 G + 4 c .. + 3 of row wrow + 8 a + g
                const unsigned p = Ds + 8u * (((2 * G + (c >> 1)) * ROWS + wrow + a * 8 + g) * 8 + 4 * (c & 1));
                const double2 v0 = qmcd_lds128s(p), v1 = qmcd_lds128s(p + 16);
                an[a][G][0][0] = v0.x; an[a][G][1][0] = v0.y; an[a][G][0][1] = v1.x; an[a][G][1][1] = v1.y;
            }
        double2 x0[2][2], x1[2][2];                                                  // [buffer][G]
#pragma unroll
        for (int G = 0; G < 2; ++G) {
            x0[0][G] = qmcd_lds128s(Ws + G * (1024 * NB) + sw0);
            x1[0][G] = qmcd_lds128s(Ws + G * (1024 * NB) + 128 + sw1);
        }
#pragma unroll
        for (int q = 0; q < NB; ++q) {
            const int cur = q & 1, nxt = cur ^ 1;
            if (q + 1 < NB) {
#pragma unroll
                for (int G = 0; G < 2; ++G) {
                    x0[nxt][G] = qmcd_lds128s(Ws + G * (1024 * NB) + (q + 1) * 1024 + sw0);
                    x1[nxt][G] = qmcd_lds128s(Ws + G * (1024 * NB) + (q + 1) * 1024 + 128 + sw1);
                }
            }
#pragma unroll
            for (int G = 0; G < 2; ++G)
#pragma unroll
                for (int a = 0; a < A_T; ++a) {
                    qmcd_dmma(an[a][G][0][0], an[a][G][0][1], T[a][q][0], x0[cur][G].x);
                    qmcd_dmma(an[a][G][1][0], an[a][G][1][1], T[a][q][0], x0[cur][G].y);
                }
#pragma unroll
            for (int G = 0; G < 2; ++G)
#pragma unroll
                for (int a = 0; a < A_T; ++a) {
                    qmcd_dmma(an[a][G][0][0], an[a][G][0][1], T[a][q][1], x1[cur][G].x);
                    qmcd_dmma(an[a][G][1][0], an[a][G][1][1], T[a][q][1], x1[cur][G].y);
                }
        }
        __syncwarp();
        if (lane == 0) qmcd_mbar_arrive(bar0 + 8 * NS + 8 * s);                      // every read of stage s is done
#pragma unroll
        for (int a = 0; a < A_T; ++a) {
            const int row = row0 + wrow + a * 8 + g;
            if (row < N) {
                double* d = Bw + (size_t)row * N + n0 + 4 * c;
#pragma unroll
                for (int G = 0; G < 2; ++G) {
                    qmcd_stg128(d + 16 * G, an[a][G][0][0], an[a][G][1][0]);
                    qmcd_stg128(d + 16 * G + 2, an[a][G][0][1], an[a][G][1][1]);
                }
            }
        }
    }
    itc = it0 + (unsigned)total;
}
