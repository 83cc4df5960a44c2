// rank_k3m_kernel -- the weighted Hermitian rank-K update of rank_k.cuh (Eq. 17 / Eq. 20; Table 1
// step 11) with the complex product taken by the 3-multiplication (Karatsuba / "3M") rule instead of its
// 4-multiplication real view.  With n_p(g) = a + i b (row operand), n_p(g') = c + i d (column operand):
//   n_p(g) conj(n_p(g')) = (a c + b d) + i (b c - a d),
//   P1 = sum_p w_p a c,   P2 = sum_p w_p b d,   P3 = sum_p w_p (a + b)(c - d)
//   Re S += P1 + P2,      Im S += P3 - P1 + P2,
// and because the row and column operands are the same vectors, all three products are needed on the lower triangle
// only.  That is 3 real DMMA contractions with k = pairs instead of 2 with k = 2 pairs: 3/4 of the tensor-pipe work
// for the same result (the cancellation in Im S is against terms of the size of |S|, i.e. an absolute error of a few
// ulp of |S|, far inside the 1e-10 relative Frobenius tolerance of the path).
//
// One CTA = one 64 x 64 complex tile of the lower triangle, ONE frequency; 8 consumer warps, each 32 rows x 16 columns
// (3 x 4 x 2 DMMA accumulators = 96 registers) + a TMA producer warp with a 3-stage ring of 32-pair chunks.  A DMMA
// k-step covers 4 pairs; a lane loads its (row, pair) / (column, pair) element with one LDS.128 (row pitch = 32 mod
// 128 bytes: the 8 lanes of a quarter-warp hit 8 distinct 16-byte bank groups) and forms a + b, w c, w d, w (c - d)
// on the FP64 ALU (10 operations per 24 DMMA).
#pragma once
#include "rank_k.cuh"

namespace rk3 {
constexpr int T = 64;
constexpr int KC = 32;                      // pairs per stage
constexpr int STAGES = 3;
#ifndef RK3_MI
#define RK3_MI 4
#endif
constexpr int MI = RK3_MI;                  // 8-row blocks per warp: warp tile (8 MI) x 16
constexpr int CONSUMER_WARPS = 4 * (T / (8 * MI));
constexpr int THREADS = (CONSUMER_WARPS + 1) * 32;
constexpr int PITCH = T * 16 + 32;          // bytes per pair row (= 32 mod 128)
constexpr int TILE_BYTES = KC * PITCH;      // 16896
constexpr int W_BYTES = KC * 8;
constexpr int STAGE_BYTES = 2 * TILE_BYTES + W_BYTES;
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 2 * STAGES * 8;
}  // namespace rk3

// Nb[Kpad][ldn] (rows >= K zero), w[n_omega][ldw], S[n_omega][ng][ldS] (lower triangle accumulated), Kpad % 32 == 0.
// Work items (tile, frequency) are numbered item = iw * ntiles + tile; grid = (n_items_of_this_launch, 1, ksplit), the
// launch covers items item_off .. item_off + gridDim.x - 1; ksplit as in rank_k_kernel (atomic tile adds when > 1).
// The host issues the whole waves with ksplit = 1 and the last partial wave K-sliced so that it also fills the GPU.
__global__ void __launch_bounds__(rk3::THREADS, 1)
rank_k3m_kernel(const cd *__restrict__ Nb, int64_t ldn, int Kpad, const double *__restrict__ w, int64_t ldw,
                cd *__restrict__ S, int64_t ldS, int64_t strideS, int ng, int ntiles, int item_off) {
    using namespace rk3;
    extern __shared__ __align__(128) unsigned char rk_smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(rk_smem + STAGES * STAGE_BYTES);
    uint64_t *empty = full + STAGES;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int item = item_off + (int)blockIdx.x;
    const int iw = item / ntiles, t = item - iw * ntiles;
    int ti = (int)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
    while ((ti + 1) * (ti + 2) / 2 <= t) ti++;
    while (ti * (ti + 1) / 2 > t) ti--;
    const int tj = t - ti * (ti + 1) / 2;
    const int row0 = ti * T, col0 = tj * T;
    const uint32_t rowbytes = (uint32_t)min(T, ng - row0) * 16u, colbytes = (uint32_t)min(T, ng - col0) * 16u;
    const uint32_t stage_tx = KC * (rowbytes + colbytes) + KC * 8u;

    // zero the ring once so that the never-copied tail columns of edge tiles hold finite numbers
    for (int i = tid; i < STAGES * STAGE_BYTES / 16; i += THREADS)
        reinterpret_cast<double2 *>(rk_smem)[i] = make_double2(0.0, 0.0);
    if (tid == 0) {
        for (int s = 0; s < STAGES; s++) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], CONSUMER_WARPS);
        }
        mbar_fence_init();
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();

    const int nk_all = Kpad / KC, ksplit = (int)gridDim.z;
    const int it0 = (int)(((int64_t)nk_all * blockIdx.z) / ksplit), it1 = (int)(((int64_t)nk_all * (blockIdx.z + 1)) / ksplit);
    const int nk = it1 - it0;
    if (warp == CONSUMER_WARPS) {
        // ---- producer warp: one 16-byte-aligned bulk copy per pair row and operand, plus the 16 weights ------------
        for (int it = 0; it < nk; it++) {
            const int s = it % STAGES;
            if (it >= STAGES) mbar_wait(&empty[s], ((it / STAGES) - 1) & 1);
            unsigned char *st = rk_smem + s * STAGE_BYTES;
            if (lane == 0) mbar_arrive_expect_tx(&full[s], stage_tx);
            __syncwarp();
            const cd *Nw = Nb + ((size_t)(it0 + it) * KC + lane) * ldn;   // KC = 32: one pair row per lane
            bulk_g2s(st + lane * PITCH, Nw + row0, rowbytes, &full[s]);
            bulk_g2s(st + TILE_BYTES + lane * PITCH, Nw + col0, colbytes, &full[s]);
            if (lane == 0) bulk_g2s(st + 2 * TILE_BYTES, w + (size_t)iw * ldw + (size_t)(it0 + it) * KC, KC * 8, &full[s]);
        }
        return;
    }

    const int g = lane >> 2, kq = lane & 3;
    const int rowoff = (warp >> 2) * (8 * MI), coloff = (warp & 3) * 16;
    // a warp whose sub-tile lies strictly above the diagonal, or wholly beyond the matrix edge (ragged last tile row /
    // column), only keeps the barriers moving: the warp sharing its scheduler then has the tensor pipe to itself
    const bool active = !(ti == tj && coloff > rowoff + 8 * MI - 1) && row0 + rowoff < ng && col0 + coloff < ng;

    double p1[MI][2][2], p2[MI][2][2], p3[MI][2][2];
#pragma unroll
    for (int mi = 0; mi < MI; mi++)
#pragma unroll
        for (int ni = 0; ni < 2; ni++)
#pragma unroll
            for (int e = 0; e < 2; e++) p1[mi][ni][e] = p2[mi][ni][e] = p3[mi][ni][e] = 0.0;

    // 8-row blocks of this warp's sub-tile that hold matrix rows (ragged last tile row): the others are skipped
    const int mi_valid = min(MI, (ng - (row0 + rowoff) + 7) / 8);
    const uint32_t a_off = kq * PITCH + (rowoff + g) * 16;
    const uint32_t b_off = TILE_BYTES + kq * PITCH + (coloff + g) * 16;
    const uint32_t w_off = 2 * TILE_BYTES + kq * 8;

    for (int it = 0; it < nk; it++) {
        const int s = it % STAGES;
        mbar_wait(&full[s], (it / STAGES) & 1);
        if (active) {
            const unsigned char *st = rk_smem + s * STAGE_BYTES;
#pragma unroll
            for (int ks = 0; ks < KC / 4; ks++) {
                const uint32_t ko = ks * 4 * PITCH;
                const double wv = *reinterpret_cast<const double *>(st + w_off + ks * 32);
                double are[MI], aim[MI], asum[MI], bre[2], bim[2], bdif[2];
#pragma unroll
                for (int mi = 0; mi < MI; mi++) {
                    const cd a = *reinterpret_cast<const cd *>(st + a_off + ko + mi * 128);
                    are[mi] = a.x;
                    aim[mi] = a.y;
                    asum[mi] = a.x + a.y;
                }
#pragma unroll
                for (int ni = 0; ni < 2; ni++) {
                    const cd b = *reinterpret_cast<const cd *>(st + b_off + ko + ni * 128);
                    bre[ni] = wv * b.x;
                    bim[ni] = wv * b.y;
                    bdif[ni] = bre[ni] - bim[ni];
                }
#pragma unroll
                for (int mi = 0; mi < MI; mi++) {
                    if (mi < mi_valid) {   // warp-uniform
#pragma unroll
                        for (int ni = 0; ni < 2; ni++) {
                            dmma(p1[mi][ni][0], p1[mi][ni][1], are[mi], bre[ni]);
                            dmma(p2[mi][ni][0], p2[mi][ni][1], aim[mi], bim[ni]);
                            dmma(p3[mi][ni][0], p3[mi][ni][1], asum[mi], bdif[ni]);
                        }
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
    }

    if (!active) return;
    cd *Sw = S + (size_t)iw * strideS;
#pragma unroll
    for (int mi = 0; mi < MI; mi++) {
        const int r = row0 + rowoff + mi * 8 + g;
        if (r >= ng) continue;
#pragma unroll
        for (int ni = 0; ni < 2; ni++) {
            const int cc = col0 + coloff + ni * 8 + 2 * kq;
#pragma unroll
            for (int e = 0; e < 2; e++) {
                const int col = cc + e;
                if (col < ng && col <= r) {
                    const double re = p1[mi][ni][e] + p2[mi][ni][e];
                    const double im = (p3[mi][ni][e] - p1[mi][ni][e]) + p2[mi][ni][e];
                    cd *ptr = Sw + (size_t)r * ldS + col;
                    if (ksplit > 1) {   // several CTAs add into this tile
                        atomicAdd(&ptr->x, re);
                        atomicAdd(&ptr->y, im);
                    } else {
                        cd v = *ptr;
                        v.x += re;
                        v.y += im;
                        *ptr = v;
                    }
                }
            }
        }
    }
}
