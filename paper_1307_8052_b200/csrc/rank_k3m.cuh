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
// One CTA = one 64 x 64 complex tile of the lower triangle, ONE frequency; EIGHT warps, all of them consumers, each
// 32 rows x 16 columns (3 x 4 x 2 DMMA accumulators = 96 registers).  A DMMA k-step covers 4 pairs; a lane loads its
// (row, pair) / (column, pair) element with one LDS.128 (row pitch = 32 mod 128 bytes: the 8 lanes of a quarter-warp hit
// 8 distinct 16-byte bank groups) and forms w c, w d, w (c - d) on the FP64 ALU (6 operations per 24 DMMA).  The row
// operand's a + b comes ready-made from a third plane, NS[pair][g] = Re + Im of N (rk3_rowsum_kernel, one pass over N per
// batch): an FP64-ALU instruction interleaved with DMMAs costs the shared FP64 datapath about three times its nominal two
// cycles (timing experiment, profiles/r2c_rank_k3m.md: -4.6 % without the four additions per k-step), an LDS.64 does not.
//
// Why eight warps and no producer warp (round 2).  The SM's register file is split over its four schedulers, so a CTA of
// nine warps (8 consumers + a TMA producer, round 1) puts three warps on one scheduler and caps EVERY thread at 168
// registers; with 96 accumulator registers that left no room to fetch the operands of the next k-step early, and ncu
// (profiles/r2c_rank_k3m.md) showed the result: the two warps of a scheduler interleave their 24 DMMAs one to one, finish
// together, and both sit in their LDS + operand-preparation bubble while the tensor pipe idles (DMMA sub-pipe 83.7 %
// busy, top stall samples on the operand-preparation instructions).  With exactly eight warps the cap is 255 registers:
// the operands of k-step ks + 1 are loaded (LDS first, preparation between the two halves of the DMMAs) into a second
// register set while the DMMAs of k-step ks issue, also across stage boundaries.  The stage refills are issued by the
// consumer warps themselves, in turn -- which is only affordable because a refill is now FOUR instructions: the row
// tile, the column tile and the row-sum tile of a 16-pair chunk are one cp.async.bulk.tensor each (2-D tensor maps over
// the N and NS buffers, boxes 16 pairs x 66 G / 68 doubles: the extra columns give the 1056- / 544-byte row pitches the
// bank-conflict-free LDS patterns need, and out-of-range columns of ragged edge tiles arrive as zeros), plus one bulk copy
// of the 16 weights.  (One 1-KB bulk copy per pair row and operand, 65 per 32-pair chunk, kept the round-1 producer warp
// 2/3 busy just issuing them: measured 60 cycles per copy; folded into the consumers that cost 25 % of the kernel.)
// Chunks of 16 pairs in a ring of 5 (213 KB) instead of 32 in a ring of 3: the third plane would not fit otherwise.
#pragma once
#include <cuda.h>
#include <algorithm>
#include <vector>
#include "rank_k.cuh"

namespace rk3 {
constexpr int T = 64;
constexpr int KC = 16;                      // pairs per stage
constexpr int STAGES = 5;
constexpr int MI = 4;                       // 8-row blocks per warp: warp tile 32 x 16 (64 x 8 measured: +1 % on configs[1] / [3], -7 % on the small matrices of configs[2])
constexpr int WARPS = 4 * (T / (8 * MI));   // 8
constexpr int THREADS = WARPS * 32;
constexpr int PITCH = T * 16 + 32;          // bytes per pair row (= 32 mod 128)
constexpr int BOX_DOUBLES = PITCH / 8;      // inner extent of the tensor-map box over N: 66 complex = 132 doubles
constexpr int TILE_BYTES = KC * PITCH;      // 16896
constexpr int SPITCH = T * 8 + 32;          // bytes per pair row of the row-sum tile (= 32 mod 128: conflict-free LDS.64)
constexpr int SBOX_DOUBLES = SPITCH / 8;    // 68
constexpr int STILE_BYTES = KC * SPITCH;    // 8704
constexpr int W_BYTES = KC * 8;
constexpr int STAGE_BYTES = 2 * TILE_BYTES + STILE_BYTES + W_BYTES;   // 42624
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 2 * STAGES * 8;
static_assert(WARPS == 8, "eight warps = 255 registers per thread");
static_assert(TILE_BYTES % 128 == 0 && STILE_BYTES % 128 == 0 && STAGE_BYTES % 128 == 0, "TMA destinations are 128-byte aligned");
static_assert(KC % 8 == 0 && KC / 4 >= 4 && (KC / 4) % 2 == 0, "k-steps of a chunk come in pairs, at least two pairs");

// operands of one k-step (4 pairs) of a warp: as loaded, and ready for the DMMAs
struct Raw {
    cd a[MI], b[2];
    double s[MI], wv;
};
struct Operands {
    double are[MI], aim[MI], asum[MI], bre[2], bim[2], bdif[2];
};
}  // namespace rk3

// Work of tile t = ti (ti + 1) / 2 + tj in 8-row x 16-column warp blocks, by the rules of rank_k3m_kernel (warps above the
// diagonal or beyond the matrix idle, diagonal tiles skip their blocks above the diagonal, ragged last rows), and the
// tiles in order of decreasing work (ties: ascending index, so that neighbours in the triangle stay neighbours).
static inline int rk3_tile_units(int ti, int tj, int ng) {
    using namespace rk3;
    const int row0 = ti * T, col0 = tj * T;
    int units = 0;
    for (int w = 0; w < WARPS; w++) {
        const int rowoff = (w >> 2) * (8 * MI), coloff = (w & 3) * 16;
        if ((ti == tj && coloff > rowoff + 8 * MI - 1) || row0 + rowoff >= ng || col0 + coloff >= ng) continue;
        const int mi_valid = std::min(MI, (ng - (row0 + rowoff) + 7) / 8);
        const int mi_lo = ti == tj ? std::max(0, (coloff - rowoff) / 8) : 0;
        units += std::max(0, mi_valid - mi_lo);
    }
    return units;
}
static inline std::vector<int32_t> rk3_tile_order(int ng) {
    const int nt = (ng + rk3::T - 1) / rk3::T;
    std::vector<int32_t> order, work;
    for (int ti = 0; ti < nt; ti++)
        for (int tj = 0; tj <= ti; tj++) {
            order.push_back(ti * (ti + 1) / 2 + tj);
            work.push_back(rk3_tile_units(ti, tj, ng));
        }
    std::stable_sort(order.begin(), order.end(), [&](int32_t a, int32_t b) { return work[a] > work[b]; });
    return order;
}

// 2-D tiled bulk tensor copy global -> shared (TMA, UTMALDG in SASS): box of the tensor map at element coordinates (x, y)
__device__ __forceinline__ void tma_load_2d(void *dst_smem, const CUtensorMap *map, int x, int y, uint64_t *bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(smem_u32(dst_smem)), "l"(map), "r"(x), "r"(y), "r"(smem_u32(bar)) : "memory");
}

// NS[p][g] = Re N[p][g] + Im N[p][g] for p < rows, g < ldn: the third operand plane of the 3M product.
// grid (rows, ceil(ldn / 256)), block 256.
__global__ void __launch_bounds__(256) rk3_rowsum_kernel(const cd *__restrict__ Nb, int64_t ldn, double *__restrict__ NS) {
    const int g = blockIdx.y * 256 + threadIdx.x;
    if (g >= ldn) return;
    const cd v = Nb[(size_t)blockIdx.x * ldn + g];
    NS[(size_t)blockIdx.x * ldn + g] = v.x + v.y;
}

// Nb[Kpad][ldn] (rows >= K zero) through nmap: a 2-D FP64 tensor map over it, dims (2 ldn, Kmax), box (132, 16); its row
// sums NS[Kpad][ldn] through smap: dims (ldn, Kmax), box (68, 16);
// w[n_omega][ldw], S[n_omega][ng][ldS] (lower triangle accumulated), Kpad % 16 == 0.
// Work items (tile, frequency) are numbered item = slot * n_omega + iw, tile = order[slot]; grid = (n_items_of_this_launch, 1, ksplit), the
// launch covers items item_off .. item_off + gridDim.x - 1; ksplit as in rank_k_kernel (atomic tile adds when > 1).
// The host issues the whole waves with ksplit = 1 and the last partial wave K-sliced so that it also fills the GPU.
__global__ void __launch_bounds__(rk3::THREADS, 1)
rank_k3m_kernel(const __grid_constant__ CUtensorMap nmap, const __grid_constant__ CUtensorMap smap, int Kpad,
                const double *__restrict__ w, int64_t ldw,
                cd *__restrict__ S, int64_t ldS, int64_t strideS, int ng, int n_omega, int item_off,
                const int32_t *__restrict__ order) {
    using namespace rk3;
    extern __shared__ __align__(128) unsigned char rk_smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(rk_smem + STAGES * STAGE_BYTES);
    uint64_t *empty = full + STAGES;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int item = item_off + (int)blockIdx.x;
    // tile-major, heaviest tiles first (order[] from rk3_tile_order): the grid's CTAs start in item order, so the light
    // tiles of the diagonal and of the ragged last row fill the end of the launch instead of leaving SMs idle behind full
    // tiles, and the n_omega CTAs of a tile run together and share its operand tiles in L2
    const int slot = item / n_omega, iw = item - slot * n_omega;
    const int t = order[slot];
    int ti = (int)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
    while ((ti + 1) * (ti + 2) / 2 <= t) ti++;
    while (ti * (ti + 1) / 2 > t) ti--;
    const int tj = t - ti * (ti + 1) / 2;
    const int row0 = ti * T, col0 = tj * T;
    constexpr uint32_t stage_tx = 2 * TILE_BYTES + STILE_BYTES + KC * 8u;   // three whole boxes (out-of-range parts arrive as zeros) + weights
    if (tid == 0) {
        for (int s = 0; s < STAGES; s++) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], WARPS);
        }
        mbar_fence_init();
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();

    const int nk_all = Kpad / KC, ksplit = (int)gridDim.z;
    const int it0 = (int)(((int64_t)nk_all * blockIdx.z) / ksplit), it1 = (int)(((int64_t)nk_all * (blockIdx.z + 1)) / ksplit);
    const int nk = it1 - it0;

    // chunk `it` of this CTA's K slice -> its ring slot: the row tile, the column tile and the row-sum tile as one tensor
    // copy each, plus the weights.  Called by one lane.
    auto refill = [&](int it) {
        const int s = it % STAGES;
        unsigned char *st = rk_smem + s * STAGE_BYTES;
        mbar_arrive_expect_tx(&full[s], stage_tx);
        tma_load_2d(st, &nmap, 2 * row0, (it0 + it) * KC, &full[s]);
        tma_load_2d(st + TILE_BYTES, &nmap, 2 * col0, (it0 + it) * KC, &full[s]);
        tma_load_2d(st + 2 * TILE_BYTES, &smap, row0, (it0 + it) * KC, &full[s]);
        bulk_g2s(st + 2 * TILE_BYTES + STILE_BYTES, w + (size_t)iw * ldw + (size_t)(it0 + it) * KC, KC * 8, &full[s]);
    };
    if (warp < STAGES && warp < nk && lane == 0) refill(warp);   // the first chunks: warps 0 .. STAGES-1

    const int g = lane >> 2, kq = lane & 3;
    const int rowoff = (warp >> 2) * (8 * MI), coloff = (warp & 3) * 16;
    // a warp whose sub-tile lies strictly above the diagonal, or wholly beyond the matrix edge (ragged last tile row /
    // column), only keeps the barriers moving and takes its refill turns: the warp sharing its scheduler then has the
    // tensor pipe to itself
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
    // ... and, in a tile on the diagonal, the 8-row blocks that lie wholly above this warp's first column
    const int mi_lo = ti == tj ? max(0, (coloff - rowoff) / 8) : 0;
    const uint32_t a_off = kq * PITCH + (rowoff + g) * 16;
    const uint32_t b_off = TILE_BYTES + kq * PITCH + (coloff + g) * 16;
    const uint32_t s_off = 2 * TILE_BYTES + kq * SPITCH + (rowoff + g) * 8;
    const uint32_t w_off = 2 * TILE_BYTES + STILE_BYTES + kq * 8;

    auto load_raw = [&](Raw &r, const unsigned char *st, int ks) {
        const uint32_t ko = ks * 4 * PITCH;
        r.wv = *reinterpret_cast<const double *>(st + w_off + ks * 32);
#pragma unroll
        for (int mi = 0; mi < MI; mi++) {
            r.a[mi] = *reinterpret_cast<const cd *>(st + a_off + ko + mi * 128);
            r.s[mi] = *reinterpret_cast<const double *>(st + s_off + ks * 4 * SPITCH + mi * 64);
        }
#pragma unroll
        for (int ni = 0; ni < 2; ni++) r.b[ni] = *reinterpret_cast<const cd *>(st + b_off + ko + ni * 128);
    };
    auto prep = [&](Operands &o, const Raw &r) {
#pragma unroll
        for (int mi = 0; mi < MI; mi++) {
            o.are[mi] = r.a[mi].x;
            o.aim[mi] = r.a[mi].y;
            o.asum[mi] = r.s[mi];
        }
#pragma unroll
        for (int ni = 0; ni < 2; ni++) {
            o.bre[ni] = r.wv * r.b[ni].x;
            o.bim[ni] = r.wv * r.b[ni].y;
            o.bdif[ni] = o.bre[ni] - o.bim[ni];
        }
    };
    auto mma_half = [&](const Operands &o, int half) {   // 8-row blocks 2 half, 2 half + 1
#pragma unroll
        for (int m2 = 0; m2 < MI / 2; m2++) {
            const int mi = half * (MI / 2) + m2;
            if (mi >= mi_lo && mi < mi_valid) {   // warp-uniform
#pragma unroll
                for (int ni = 0; ni < 2; ni++) {
                    dmma(p1[mi][ni][0], p1[mi][ni][1], o.are[mi], o.bre[ni]);
                    dmma(p2[mi][ni][0], p2[mi][ni][1], o.aim[mi], o.bim[ni]);
                    dmma(p3[mi][ni][0], p3[mi][ni][1], o.asum[mi], o.bdif[ni]);
                }
            }
        }
    };
    // one k-step: the loads of the next k-step first, its FP64-ALU preparation between the two halves of the DMMAs
    auto step = [&](const Operands &cur, Operands &nxt, const unsigned char *st_next, int ks_next) {
        Raw r;
        load_raw(r, st_next, ks_next);
        mma_half(cur, 0);
        prep(nxt, r);
        mma_half(cur, 1);
    };

    Operands oa, ob;
    if (nk > 0) {
        mbar_wait(&full[0], 0);
        if (active) {
            Raw r;
            load_raw(r, rk_smem, 0);
            prep(oa, r);
        }
    }
    for (int it = 0; it < nk; it++) {
        const int s = it % STAGES;
        const unsigned char *st = rk_smem + s * STAGE_BYTES;
        if (active) {
#pragma unroll
            for (int ks = 0; ks < KC / 4 - 2; ks += 2) {
                step(oa, ob, st, ks + 1);
                step(ob, oa, st, ks + 2);
            }
            step(oa, ob, st, KC / 4 - 1);   // the last k-step but one under the loads of the last: the chunk is now all in registers
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);   // release the slot
        if (it + 1 < nk) {                        // the last k-step under the loads of k-step 0 of the next chunk
            const int s1 = (it + 1) % STAGES;
            mbar_wait(&full[s1], ((it + 1) / STAGES) & 1);
            if (active) step(ob, oa, rk_smem + s1 * STAGE_BYTES, 0);
        } else if (active) {
            mma_half(ob, 0);
            mma_half(ob, 1);
        }
        // refill turn: chunk it + STAGES goes into the slot just released, once all eight warps have released it
        if (it + STAGES < nk && (it & (WARPS - 1)) == warp && lane == 0) {
            mbar_wait(&empty[s], (it / STAGES) & 1);
            refill(it + STAGES);
        }
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
