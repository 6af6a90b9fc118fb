// qmcd_flush_tma.cuh -- the rank-m flush of Eq. 4 for K <= 64, one tile of 128 rows
// of B per call, with every operand brought into shared memory by TMA (cp.async.bulk.tensor + mbarrier)
// and the eight warps doing nothing but LDS.128 + DMMA.8x8x4:
//
//     iterations 0 .. nk-1      (nk = N/32)   T  = B0[tile, 32 k-columns] . C[:, same]^T   accumulated in registers
//     iteration  nk                            T  = -T + E_J ;  T <- T M                   (M = S^-1, 64 x 64, zero outside m x m)
//     iterations nk+1 .. 2nk                   B[tile, 32 columns] += T . W[:, same]       written back from registers
//
// One ring of 3 stages of 48 KB carries all of it; stage contents per kind of iteration:
//     NT : B0 tile as [4 k-groups][128 rows][8]      + C as [4 k-groups][8 NB rows][8]          (4-D tensor maps, no swizzle:
//          an 8 x 8 fp64 fragment block is 512 contiguous bytes, so the 16-byte fragment loads are conflict-free)
//     M  : M as [4 column groups][64 rows][16]       (SWIZZLE_128B: 16-byte chunk ^= row % 8 -- with the permuted
//          contraction index k = 8q + 2c + s of qmcd_flush_mma.cuh the fragment loads are conflict-free)
//     NN : B0 tile as [4 column groups][128 rows][8] + W as [2 column groups][8 NB rows][16]   (W swizzled like M)
// A warp owns 16 rows of the tile through all three parts, so nothing but the ring's mbarriers synchronises
// the CTA.  Thread 0 issues the loads two iterations ahead (half way through an iteration it waits for the
// stage freed one iteration ago -- by then every warp has left it).  Rows past N and queue rows past K are
// zero-filled by TMA; ranks m < K use the leading mp8 = round8(m) columns / rows only.
#pragma once
#include <cuda.h>
#include "qmcd_flush_mma.cuh"

struct QmcdTmaps { CUtensorMap B, C, W, M; };      // 4-D views, see qmcd_api.cu (encode_tmaps)

#define QMCD_TMA_NS 3
#define QMCD_TMA_STAGE_BYTES 49152
#define QMCD_TMA_BAR_OFF 512                 // full[3], empty[3] mbarriers inside the shared-memory header
#define QMCD_TMA_STAGE_OFF 1024              // stages are 1024-byte aligned (swizzle atoms)
#define QMCD_TMA_LDT 72                      // row stride of T in doubles (== 8 mod 16: conflict-free fragment loads)
#define QMCD_TMA_ROWS 128
__host__ __device__ inline size_t qmcd_flush_tma_smem_bytes() {
    return (size_t)QMCD_TMA_STAGE_OFF + QMCD_TMA_NS * QMCD_TMA_STAGE_BYTES + (size_t)QMCD_TMA_ROWS * QMCD_TMA_LDT * 8;
}
__host__ __device__ inline int qmcd_tma_NB(int K) { return K <= 8 ? 1 : K <= 16 ? 2 : K <= 32 ? 4 : 8; }

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
__device__ __forceinline__ void qmcd_fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

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

// One tile.  `itc` = iterations this CTA has pushed through the ring so far (the same in every thread; it
// fixes stage and mbarrier parity), updated on return.  All 256 threads; ends without a CTA barrier.
template <int NB>
__device__ __noinline__ void qmcd_flush_tile_tma(const QmcdDev& P, const QmcdTmaps& TM, unsigned char* smem, int b, int m, int tile,
                                    unsigned& itc) {
    constexpr int NG = (NB + 1) / 2;              // 16-column groups of T
    constexpr unsigned TX_ROWS = 32768u + 2048u * NB;
    const int N = P.N, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, g = lane >> 2, c = lane & 3;
    const int mp8 = (m + 7) & ~7, nqm = mp8 >> 3, nG = (mp8 + 15) >> 4;
    const int nk = N / 32, total = 2 * nk + 1;
    const int row0 = tile * QMCD_TMA_ROWS;
    const unsigned bar0 = qmcd_su32(smem + QMCD_TMA_BAR_OFF);
    unsigned char* st0 = smem + QMCD_TMA_STAGE_OFF;
    double* Ts = reinterpret_cast<double*>(st0 + QMCD_TMA_NS * QMCD_TMA_STAGE_BYTES);
    const unsigned it0 = itc;
    double* Bw = P.B + (size_t)b * N * N;
    const int* Jw = P.J + (size_t)b * P.K;

    auto issue = [&](int j) {                     // thread 0: the loads of iteration j of this tile
        const unsigned gi = it0 + (unsigned)j, s = gi % QMCD_TMA_NS, u = gi / QMCD_TMA_NS;
        if (u > 0) qmcd_mbar_wait(bar0 + 8 * QMCD_TMA_NS + 8 * s, (u - 1) & 1);      // every warp has left the stage
        const unsigned dst = qmcd_su32(st0 + s * QMCD_TMA_STAGE_BYTES), fb = bar0 + 8 * s;
        if (j < nk) {
            qmcd_mbar_expect_tx(fb, TX_ROWS);
            qmcd_tma_load4(dst, &TM.B, 0, row0, 4 * j, b, fb);
            qmcd_tma_load4(dst + 32768, &TM.C, 0, 0, 4 * j, b, fb);
        } else if (j == nk) {
            qmcd_mbar_expect_tx(fb, 32768u);
            qmcd_tma_load4(dst, &TM.M, 0, 0, 0, b, fb);
        } else {
            const int jj = j - nk - 1;
            qmcd_mbar_expect_tx(fb, TX_ROWS);
            qmcd_tma_load4(dst, &TM.B, 0, row0, 4 * jj, b, fb);
            qmcd_tma_load4(dst + 32768, &TM.W, 0, 0, 2 * jj, b, fb);
        }
    };
    if (tid == 0) { issue(0); issue(1); }

    double acc[2][NB][2];
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int bt = 0; bt < NB; ++bt) { acc[a][bt][0] = 0.0; acc[a][bt][1] = 0.0; }
    const double* Trow = Ts + (size_t)(wid * 16 + g) * QMCD_TMA_LDT + 2 * c;     // + a * 8 * LDT + 8 q

    for (int j = 0; j < total; ++j) {
        const unsigned gi = it0 + (unsigned)j, s = gi % QMCD_TMA_NS, u = gi / QMCD_TMA_NS;
        const unsigned char* stg = st0 + s * QMCD_TMA_STAGE_BYTES;
        qmcd_mbar_wait(bar0 + 8 * s, u & 1);
        if (j < nk) {
            // ---- NT: 4 k-groups of 8 columns; fragments are 16-byte vectors (k = 8q + 2c + s on both operands)
            const double* As = reinterpret_cast<const double*>(stg) + (wid * 16 + g) * 8 + 2 * c;
            const double* Cs = reinterpret_cast<const double*>(stg + 32768) + g * 8 + 2 * c;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (q == 2 && tid == 0 && j + 2 < total) issue(j + 2);
                double2 av[2], bv[NB];
#pragma unroll
                for (int a = 0; a < 2; ++a) av[a] = qmcd_lds128(As + q * (QMCD_TMA_ROWS * 8) + a * 64);
#pragma unroll
                for (int bt = 0; bt < NB; ++bt) bv[bt] = qmcd_lds128(Cs + q * (64 * NB) + bt * 64);
#pragma unroll
                for (int bt = 0; bt < NB; ++bt)
                    if (bt < nqm) {
#pragma unroll
                        for (int a = 0; a < 2; ++a) qmcd_dmma(acc[a][bt][0], acc[a][bt][1], av[a].x, bv[bt].x);
                    }
#pragma unroll
                for (int bt = 0; bt < NB; ++bt)
                    if (bt < nqm) {
#pragma unroll
                        for (int a = 0; a < 2; ++a) qmcd_dmma(acc[a][bt][0], acc[a][bt][1], av[a].y, bv[bt].y);
                    }
            }
        } else if (j == nk) {
            if (tid == 0 && j + 2 < total) issue(j + 2);
            // ---- T = -(B0 C^T) + E_J for this warp's 16 rows, then T <- T M (warp-local)
            double* Tw = Ts + (size_t)(wid * 16 + g) * QMCD_TMA_LDT + 2 * c;
#pragma unroll
            for (int a = 0; a < 2; ++a)
#pragma unroll
                for (int bt = 0; bt < NB; ++bt)
                    if (bt < nqm)
                        *reinterpret_cast<double2*>(Tw + a * 8 * QMCD_TMA_LDT + bt * 8) = make_double2(-acc[a][bt][0], -acc[a][bt][1]);
            __syncwarp();
            for (int i = lane; i < m; i += 32) {
                const int r = __ldcg(Jw + i) - row0 - wid * 16;
                if (r >= 0 && r < 16) Ts[(size_t)(wid * 16 + r) * QMCD_TMA_LDT + i] += 1.0;
            }
            __syncwarp();
            double a2[2][NG][2][2];
#pragma unroll
            for (int a = 0; a < 2; ++a)
#pragma unroll
                for (int G = 0; G < NG; ++G) { a2[a][G][0][0] = a2[a][G][0][1] = a2[a][G][1][0] = a2[a][G][1][1] = 0.0; }
            const unsigned char* Ms = stg + (2 * c) * 128;          // row k = 8q + 2c (+1), chunk g ^ (k % 8)
            const int sw0 = (g ^ (2 * c)) << 4, sw1 = (g ^ (2 * c + 1)) << 4;
#pragma unroll
            for (int q = 0; q < NB; ++q) {
                if (q < nqm) {
                    double2 av[2];
#pragma unroll
                    for (int a = 0; a < 2; ++a) av[a] = qmcd_lds128(Trow + a * 8 * QMCD_TMA_LDT + 8 * q);
#pragma unroll
                    for (int G = 0; G < NG; ++G) {
                        if (G < nG) {
                            const double2 x0 = *reinterpret_cast<const double2*>(Ms + G * 8192 + q * 1024 + sw0);
                            const double2 x1 = *reinterpret_cast<const double2*>(Ms + G * 8192 + q * 1024 + 128 + sw1);
#pragma unroll
                            for (int a = 0; a < 2; ++a) {
                                qmcd_dmma(a2[a][G][0][0], a2[a][G][0][1], av[a].x, x0.x);
                                qmcd_dmma(a2[a][G][1][0], a2[a][G][1][1], av[a].x, x0.y);
                                qmcd_dmma(a2[a][G][0][0], a2[a][G][0][1], av[a].y, x1.x);
                                qmcd_dmma(a2[a][G][1][0], a2[a][G][1][1], av[a].y, x1.y);
                            }
                        }
                    }
                }
            }
            __syncwarp();                                // every lane has read this warp's rows of T
            double* To = Ts + (size_t)(wid * 16 + g) * QMCD_TMA_LDT + 4 * c;
#pragma unroll
            for (int a = 0; a < 2; ++a)
#pragma unroll
                for (int G = 0; G < NG; ++G)
                    if (G < nG) {                        // columns 16 G + 4 c .. + 3 (n-slot x of tile t is column 16 G + 2 x + t)
                        *reinterpret_cast<double2*>(To + a * 8 * QMCD_TMA_LDT + 16 * G) = make_double2(a2[a][G][0][0], a2[a][G][1][0]);
                        *reinterpret_cast<double2*>(To + a * 8 * QMCD_TMA_LDT + 16 * G + 2) = make_double2(a2[a][G][0][1], a2[a][G][1][1]);
                    }
            __syncwarp();
        } else {
            // ---- NN: B[tile, 32 columns] += T W[:, same]; initial values from the staged tile, results by STG
            const int n0 = 32 * (j - nk - 1);
            const double* Ds = reinterpret_cast<const double*>(stg);                 // [4 groups of 8 columns][128 rows][8]
            const unsigned char* Ws = stg + 32768 + (2 * c) * 128;                    // [2 groups of 16 columns][8 NB rows][128 B]
            const int sw0 = (g ^ (2 * c)) << 4, sw1 = (g ^ (2 * c + 1)) << 4;
            double an[2][2][2][2];
#pragma unroll
            for (int a = 0; a < 2; ++a)
#pragma unroll
                for (int G = 0; G < 2; ++G) {          // this lane's columns 16 G + 4 c .. + 3 of rows 16 wid + 8 a + g
                    const double* p = Ds + ((2 * G + (c >> 1)) * QMCD_TMA_ROWS + wid * 16 + a * 8 + g) * 8 + 4 * (c & 1);
                    const double2 v0 = qmcd_lds128(p), v1 = qmcd_lds128(p + 2);
                    an[a][G][0][0] = v0.x; an[a][G][1][0] = v0.y; an[a][G][0][1] = v1.x; an[a][G][1][1] = v1.y;
                }
#pragma unroll
            for (int q = 0; q < NB; ++q) {
                if (q == (nqm >> 1) && tid == 0 && j + 2 < total) issue(j + 2);
                if (q < nqm) {
                    double2 av[2], x0[2], x1[2];
#pragma unroll
                    for (int a = 0; a < 2; ++a) av[a] = qmcd_lds128(Trow + a * 8 * QMCD_TMA_LDT + 8 * q);
#pragma unroll
                    for (int G = 0; G < 2; ++G) {
                        x0[G] = *reinterpret_cast<const double2*>(Ws + G * (1024 * NB) + q * 1024 + sw0);
                        x1[G] = *reinterpret_cast<const double2*>(Ws + G * (1024 * NB) + q * 1024 + 128 + sw1);
                    }
#pragma unroll
                    for (int G = 0; G < 2; ++G)
#pragma unroll
                        for (int a = 0; a < 2; ++a) {
                            qmcd_dmma(an[a][G][0][0], an[a][G][0][1], av[a].x, x0[G].x);
                            qmcd_dmma(an[a][G][1][0], an[a][G][1][1], av[a].x, x0[G].y);
                        }
#pragma unroll
                    for (int G = 0; G < 2; ++G)
#pragma unroll
                        for (int a = 0; a < 2; ++a) {
                            qmcd_dmma(an[a][G][0][0], an[a][G][0][1], av[a].y, x1[G].x);
                            qmcd_dmma(an[a][G][1][0], an[a][G][1][1], av[a].y, x1[G].y);
                        }
                }
            }
#pragma unroll
            for (int a = 0; a < 2; ++a) {
                const int row = row0 + wid * 16 + a * 8 + g;
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
        __syncwarp();
        if (lane == 0) qmcd_mbar_arrive(bar0 + 8 * QMCD_TMA_NS + 8 * s);       // this warp has left stage s
    }
    itc = it0 + (unsigned)total;
}
