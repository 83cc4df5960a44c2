// Transition weights (Eq. 18, in the real form of BASELINE.json north_star) and the weighted Hermitian
// rank-K update for every imaginary frequency (Eq. 17 / Eq. 20; Table 1 step 11):
//   S_w[g][g'] += sum_{p < K} w[w][p] n_p(g) conj(n_p(g')),      g >= g' only (one triangle).
//
// FP64 tensor cores: the only native FP64 MMA on sm_100a is DMMA.8x8x4 (mma.sync.m8n8k4.f64).  The complex
// product is taken in its real view: with k = 2p + c (c = 0: re, 1: im),
//   Re S[g][g'] = sum_k  A[g][k] B[k][g'],   A[g][2p+c]  = w_p (re, im) n_p(g),   B[2p+c][g'] = (re, im) n_p(g')
//   Im S[g][g'] = sum_k A'[g][k] B[k][g'],   A'[g][2p+c] = w_p (im, -re) n_p(g)
// so one staged N tile feeds both; A and A' are the same shared-memory words read with c and c^1.  The N buffer is
// pair-major ([p][g], g contiguous) exactly as the sphere gather writes it: a DMMA fragment is then 2 pair rows x
// 8 consecutive complex numbers = 2 x 128 B.  An LDS.64 is served per half-warp (4 g values x 2 pair rows x 16 B):
// with a row pitch = 64 (mod 128) bytes the two pair rows of a half-warp fall in different bank halves.
//
// One CTA = one 64 x 64 complex tile of the lower triangle x 2 frequencies (warps 0-3: first, 4-7: second; each
// warp a 32 x 32 complex sub-tile = 4 x 4 x {Re,Im} DMMA accumulators = 128 registers).  K is streamed in chunks
// of 16 pairs through a 5-stage ring filled by a dedicated producer warp through the TMA engine (cp.async.bulk, one
// 1 KB row per copy) and tracked with full/empty mbarriers.  Both frequencies share the staged rows; only the
// weights differ, and they multiply the column operand (4 DMUL per 32 DMMA).
#pragma once
#include "common.cuh"

namespace rk {
constexpr int T = 64;        // tile edge (complex elements)
constexpr int KC = 16;       // pairs per stage
constexpr int STAGES = 5;
constexpr int PITCH = T * 16 + 64;               // bytes per pair row in shared memory (= 64 mod 128, see below)
constexpr int TILE_BYTES = KC * PITCH;           // 17408
// SHARED_N = true : the chi0 accumulation: 2 frequencies per CTA read the same N tiles; 8 consumer warps + the TMA
//                   producer warp, 5 stages, one CTA per SM (K is thousands of pairs: the ring never drains).
// SHARED_N = false: the Cholesky trailing update of rpa_ec_q: every frequency has its own N (the transposed panel of
//                   that frequency's matrix) and K is one panel (32 pairs), so a CTA is mostly prologue (TMA round
//                   trip) and epilogue (read-modify-write of its tile): 1 frequency per CTA, 4 consumer warps,
//                   2 stages (= the whole panel), two CTAs per SM so that one computes while the other loads / stores.
//                   The weights are NOT applied: this instance computes S -= N N^H (w = -1 for every pair).
template <bool SHARED_N>
struct Cfg {
    static constexpr int NW = SHARED_N ? 2 : 1;               // frequencies per CTA
    static constexpr int CONSUMER_WARPS = 4 * NW;
    static constexpr int THREADS = (CONSUMER_WARPS + 1) * 32; // the last warp is the TMA producer
    static constexpr int MIN_CTAS = SHARED_N ? 1 : 2;
    static constexpr int NSTAGES = SHARED_N ? STAGES : 2;
    static constexpr int W_BYTES = NW * KC * 8;
    static constexpr int STAGE_BYTES = 2 * TILE_BYTES + W_BYTES;
    static constexpr int SMEM_BYTES = NSTAGES * STAGE_BYTES + 2 * NSTAGES * 8;
};
}  // namespace rk

// eta < 0 (imaginary axis, Eq. 18 in its real form, reading A1):
//   w[iw*ldw + p] = kweight * 2 (f_n - f_m)(e_n - e_m) / (omega_iw^2 + (e_n - e_m)^2) for p < K, 0 for K <= p < Kpad.
// eta > 0 (real axis, NEXT-4, reading A19): slot iw = 2 i + part holds the real (part 0) or imaginary (part 1) part of
//   w = kweight (f_n - f_m) [1/(z - D) - 1/(z + D)],  z = omega_i + i eta,  D = e_m - e_n,   1/(x + i eta) = (x - i eta)/(x^2 + eta^2)
// (omega[] holds omega_i twice), so that chi0 = S(Re w) + i S(Im w) with two Hermitian accumulators.
__global__ void weights_kernel(double *__restrict__ w, int64_t ldw, int K, int Kpad, const double *__restrict__ omega,
                               int n_omega, const double *__restrict__ eps_occ, const double *__restrict__ f_occ,
                               const double *__restrict__ eps_unocc, const double *__restrict__ f_unocc, int n0,
                               int mlen, int m0, double kweight, double eta) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    const int iw = blockIdx.y;
    if (p >= Kpad || iw >= n_omega) return;
    double val = 0.0;
    if (p < K) {
        const int n = n0 + p / mlen, m = m0 + p % mlen;
        const double de = eps_occ[n] - eps_unocc[m];
        const double om = omega[iw];
        const double df = f_occ[n] - f_unocc[m];
        if (eta < 0.0) {
            val = kweight * (2.0 * df * de / (om * om + de * de));
        } else {
            const double xm = om + de, xp = om - de;   // z - D and z + D without the i eta
            const double dm = xm * xm + eta * eta, dp = xp * xp + eta * eta;
            val = (iw & 1) ? kweight * df * (eta / dp - eta / dm) : kweight * df * (xm / dm - xp / dp);
        }
    }
    w[(size_t)iw * ldw + p] = val;
}

// Nb[Kpad][ldn] (rows >= K are zero; frequency iw reads Nb + iw*strideN, strideN = 0 when SHARED_N), w[n_omega][ldw],
// S[n_omega][ng][ldS] (lower triangle accumulated).  Only rows / columns g >= g0 are touched (g0 % 1 == 0; tiles
// start at g0).  Kpad % KC == 0.  grid = (tiles selected by tile_mode, ceil(n_omega / Cfg::NW), ksplit).
// ksplit > 1 (chi0 accumulation only): CTA z takes the z-th slice of the K chunks and adds its tile with
// red.global.add.f64, so that tiles x frequency pairs x slices fill the last wave of the grid (the host picks
// ksplit); the order of those additions is not fixed, i.e. S is then reproducible to rounding, not bitwise.
template <bool SHARED_N>
__global__ void __launch_bounds__(rk::Cfg<SHARED_N>::THREADS, rk::Cfg<SHARED_N>::MIN_CTAS)
rank_k_kernel(const cd *__restrict__ Nb, int64_t ldn, int64_t strideN, int Kpad, const double *__restrict__ w,
              int64_t ldw, cd *__restrict__ S, int64_t ldS, int64_t strideS, int ng, int g0, int n_omega,
              int tile_mode, int col_limit) {
    using namespace rk;
    constexpr int STAGES = Cfg<SHARED_N>::NSTAGES;
    constexpr int STAGE_BYTES = Cfg<SHARED_N>::STAGE_BYTES;
    constexpr int NW = Cfg<SHARED_N>::NW, CONSUMER_WARPS = Cfg<SHARED_N>::CONSUMER_WARPS, THREADS = Cfg<SHARED_N>::THREADS;
    constexpr int W_OFF = 2 * TILE_BYTES;
    extern __shared__ __align__(128) unsigned char rk_smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(rk_smem + STAGES * STAGE_BYTES);
    uint64_t *empty = full + STAGES;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // lower-triangle tile (ti >= tj) from the linear index
    // tile_mode 0: all lower tiles; 1: only the first tile column (tj = 0, blockIdx.x = ti); 2: all the others
    // (the lower tiles of the triangle shifted by one tile); 3: the first two tile columns; 4: all the others (shifted by
    // two tiles) -- the blocked Cholesky of rpa_ec_q uses 1 (strips), 3 and 4.
    // Columns >= col_limit (<= ng) are not written (a strip update inside a Cholesky block touches one 32-column panel).
    const int t = blockIdx.x;
    int ti, tj;
    if (tile_mode == 1) {
        ti = t;
        tj = 0;
    } else if (tile_mode == 3) {
        const int nt = (ng - g0 + T - 1) / T;
        ti = t < nt ? t : t - nt + 1;
        tj = t < nt ? 0 : 1;
    } else {
        ti = (int)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
        while ((ti + 1) * (ti + 2) / 2 <= t) ti++;
        while (ti * (ti + 1) / 2 > t) ti--;
        tj = t - ti * (ti + 1) / 2;
        if (tile_mode == 2) { ti++; tj++; }
        if (tile_mode == 4) { ti += 2; tj += 2; }
    }
    const int row0 = g0 + ti * T, col0 = g0 + tj * T;
    const int om0 = blockIdx.y * NW;
    const int n_om = min(NW, n_omega - om0);
    const uint32_t rowbytes = (uint32_t)min(T, ng - row0) * 16u, colbytes = (uint32_t)min(T, ng - col0) * 16u;
    const uint32_t stage_tx = KC * (rowbytes + colbytes) + (uint32_t)n_om * KC * 8u;

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

    // this CTA's slice of the K chunks
    const int nk_all = Kpad / KC, ksplit = (int)gridDim.z;
    const int it0 = (int)(((int64_t)nk_all * blockIdx.z) / ksplit), it1 = (int)(((int64_t)nk_all * (blockIdx.z + 1)) / ksplit);
    const int nk = it1 - it0;
    if (warp == CONSUMER_WARPS) {
        // ---- producer warp: keeps the ring full, never touches the tensor pipe -------------------------------
        for (int it = 0; it < nk; it++) {
            const int s = it % STAGES;
            if (it >= STAGES) mbar_wait(&empty[s], ((it / STAGES) - 1) & 1);
            unsigned char *st = rk_smem + s * STAGE_BYTES;
            if (lane == 0) mbar_arrive_expect_tx(&full[s], stage_tx);
            __syncwarp();
            const size_t krow = (size_t)(it0 + it) * KC + (lane & 15);
            const cd *Nw = Nb + (size_t)om0 * strideN + krow * ldn;   // strideN = 0 when SHARED_N
            if (lane < 16) bulk_g2s(st + lane * PITCH, Nw + row0, rowbytes, &full[s]);
            else bulk_g2s(st + TILE_BYTES + (lane - 16) * PITCH, Nw + col0, colbytes, &full[s]);
            if (lane < n_om)
                bulk_g2s(st + W_OFF + lane * KC * 8, w + (size_t)(om0 + lane) * ldw + (size_t)(it0 + it) * KC, KC * 8, &full[s]);
        }
        return;
    }

    const int g = lane >> 2, kq = lane & 3, pp = kq >> 1, c = kq & 1;
    const int wsel = warp >> 2, quad = warp & 3;
    const int rowoff = (quad >> 1) * 32, coloff = (quad & 1) * 32;
    // a warp whose sub-tile lies strictly above the diagonal, wholly beyond the matrix edge or the column limit, or whose
    // frequency does not exist, only keeps the barriers moving
    // (col_limit: a Cholesky strip update writes only 32 of the tile's 64 columns)
    const bool active = (wsel < n_om) && !(ti == tj && coloff > rowoff) && row0 + rowoff < ng && col0 + coloff < min(ng, col_limit);

    if (!SHARED_N && active) {   // short K: pull this warp's part of the accumulator tile towards L2 while the K loop runs
        const cd *Sp = S + (size_t)(om0 + wsel) * strideS;
#pragma unroll
        for (int i = 0; i < 4; i++) {
            const int r = row0 + rowoff + i * 8 + g, cc = col0 + coloff + kq * 8;
            if (r < ng && cc < ng && cc <= r) asm volatile("prefetch.global.L2 [%0];" ::"l"(Sp + (size_t)r * ldS + cc));
        }
    }

    double re[4][4][2], im[4][4][2];
#pragma unroll
    for (int mi = 0; mi < 4; mi++)
#pragma unroll
        for (int ni = 0; ni < 4; ni++) re[mi][ni][0] = re[mi][ni][1] = im[mi][ni][0] = im[mi][ni][1] = 0.0;

    const uint32_t a_off = pp * PITCH + (rowoff + g) * 16;
    const uint32_t b_off = TILE_BYTES + pp * PITCH + (coloff + g) * 16 + c * 8;
    const uint32_t w_off = W_OFF + (wsel * KC + pp) * 8;
    const uint32_t sign_hi = (uint32_t)c << 31;   // A'[2p+1] = -re: flip the sign bit on odd k lanes (ALU pipe, not FP64)

    for (int it = 0; it < nk; it++) {
        const int s = it % STAGES;
        mbar_wait(&full[s], (it / STAGES) & 1);
        if (active) {
            const unsigned char *st = rk_smem + s * STAGE_BYTES;
#pragma unroll
            for (int ks = 0; ks < KC / 2; ks++) {
                const uint32_t ko = ks * 2 * PITCH;
                // the weight multiplies the shared (column) operand: 4 DMUL per k-step instead of 8
                const double wv = *reinterpret_cast<const double *>(st + w_off + ks * 16);
                double a[4], a2[4], b[4];
#pragma unroll
                for (int mi = 0; mi < 4; mi++) {
                    const unsigned char *ap = st + a_off + ko + mi * 128;
                    a[mi] = *reinterpret_cast<const double *>(ap + c * 8);
                    const double o = *reinterpret_cast<const double *>(ap + (c ^ 1) * 8);
                    a2[mi] = __hiloint2double(__double2hiint(o) ^ (int)sign_hi, __double2loint(o));
                }
#pragma unroll
                for (int ni = 0; ni < 4; ni++) {
                    const double bv = *reinterpret_cast<const double *>(st + b_off + ko + ni * 128);
                    // the Cholesky update's weight is -1 for every pair: taken as the subtraction in the epilogue, which saves
                    // the four FP64 multiplications per k-step on the datapath the DMMAs share (same bits: the sums are negated)
                    b[ni] = SHARED_N ? wv * bv : bv;
                }
#pragma unroll
                for (int mi = 0; mi < 4; mi++)
#pragma unroll
                    for (int ni = 0; ni < 4; ni++) {
                        dmma(re[mi][ni][0], re[mi][ni][1], a[mi], b[ni]);
                        dmma(im[mi][ni][0], im[mi][ni][1], a2[mi], b[ni]);
                    }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
    }

    if (!active) return;
    cd *Sw = S + (size_t)(om0 + wsel) * strideS;
    if constexpr (SHARED_N) {
        // long K: the epilogue is < 1 % of the CTA; plain read-modify-write keeps the register count of the K loop
#pragma unroll
        for (int mi = 0; mi < 4; mi++) {
            const int r = row0 + rowoff + mi * 8 + g;
            if (r >= ng) continue;
#pragma unroll
            for (int ni = 0; ni < 4; ni++) {
                const int cc = col0 + coloff + ni * 8 + 2 * kq;
#pragma unroll
                for (int e = 0; e < 2; e++) {
                    const int col = cc + e;
                    if (col < col_limit && col <= r) {
                        cd *ptr = Sw + (size_t)r * ldS + col;
                        if (ksplit > 1) {   // several CTAs add into this tile
                            atomicAdd(&ptr->x, re[mi][ni][e]);
                            atomicAdd(&ptr->y, im[mi][ni][e]);
                        } else {
                            cd v = *ptr;
                            v.x += re[mi][ni][e];
                            v.y += im[mi][ni][e];
                            *ptr = v;
                        }
                    }
                }
            }
        }
    } else {
        // short K: the read-modify-write is a large part of the CTA: all loads of an 8-row group are issued before
        // its stores (a CTA owns its tile, but the compiler cannot know that the pointers do not alias)
#pragma unroll
        for (int mi = 0; mi < 4; mi++) {
            const int r = row0 + rowoff + mi * 8 + g;
            if (r >= ng) continue;
            cd *rowp = Sw + (size_t)r * ldS;
            cd v[4][2];
#pragma unroll
            for (int ni = 0; ni < 4; ni++) {
                const int cc = col0 + coloff + ni * 8 + 2 * kq;
#pragma unroll
                for (int e = 0; e < 2; e++)
                    if (cc + e < col_limit && cc + e <= r) v[ni][e] = rowp[cc + e];
            }
#pragma unroll
            for (int ni = 0; ni < 4; ni++) {
                const int cc = col0 + coloff + ni * 8 + 2 * kq;
#pragma unroll
                for (int e = 0; e < 2; e++)
                    if (cc + e < col_limit && cc + e <= r) {
                        v[ni][e].x -= re[mi][ni][e];
                        v[ni][e].y -= im[mi][ni][e];
                        rowp[cc + e] = v[ni][e];
                    }
            }
        }
    }
}
