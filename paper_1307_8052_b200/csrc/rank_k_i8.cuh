// rank_k_i8 -- the weighted Hermitian rank-K update of rank_k3m.cuh (Eq. 17 / Eq. 20) on the INT8
// tensor pipe (tcgen05.mma.kind::i8, s32 accumulators in TMEM) by error-free slicing (the Ozaki scheme).
//
// Real form of one frequency: with n_p(g) = a + i b,
//   Re S[g][g'] = sum_p (a_g)(w a_g') + (b_g)(w b_g'),     Im S[g][g'] = sum_p (b_g)(w a_g') + (-a_g)(w b_g'),
// i.e. D = L R^T with L = [a | b ; b | -a] (2 ngp "left rows", K' = 2 Kpad columns) and R_w = [w a | w b] (ng rows).
// Every row of L is scaled by a power of two to (-1, 1) and cut into I8_S signed digits
//   x = sum_i d_i 2^(-6 - 7 i) + r,   d_i in [-64, 64],   |r| <= 2^(-7 - 7 (S - 1))   (one rounding to 6 + 7 (S - 1) bits),
// likewise every row of R_w (scaled per frequency and row).  The digit products L_i R_j^T with i + j = t share the
// scale 2^(-12 - 7 t); each t has its own s32 accumulator in TMEM (exact: at most S * K' * 64^2 < 2^31), the pairs with
// i + j >= S are below the truncation error and are dropped.  The epilogue recombines in FP64:
//   D = 2^eL[g] 2^eR[g'] 2^-12 sum_t 2^(-7 t) P_t    -> added to S (real part for the upper half of L, imaginary for the lower).
//
// Operand reuse: a CTA owns a 128 x 64 tile of D.  Per 32-column K block it stages ALL digits of its rows and columns
// once (S x 4 KB + S x 2 KB, packed by the slicing kernels in exactly the shared-memory layout of the MMA: K-major,
// no swizzle, 8-row x 16-byte core matrices) with two bulk copies and issues the S (S + 1) / 2 MMAs of 128 x 64 x 32.
#pragma once
#include "rank_k.cuh"
#include "probe_i8.cuh"

namespace rki8 {
// S = digits per operand: 6 + 7 (S - 1) bits of the row's power-of-two scale.  S = 7 (48 bits): agrees with the FP64 tensor
// path to ~1e-14 relative Frobenius; S = 6 (41 bits): ~3e-12, 3/4 of the MMAs; S = 8 (55 bits: every element within 2^-2 of
// its row maximum is sliced without any rounding; 36 digit products instead of 28, all 512 TMEM columns).
constexpr int RB = 128, CB = 64;     // rows / columns of a CTA tile
constexpr int KB = 32;               // K' entries (bytes) per MMA
constexpr int A_BYTES = RB * KB, B_BYTES = CB * KB;
constexpr int STAGES = 4;
__host__ __device__ constexpr int stage_bytes(int S) { return S * (A_BYTES + B_BYTES); }   // 36864 (S = 6), 43008 (S = 7)
__host__ __device__ constexpr int smem_bytes(int S) { return STAGES * stage_bytes(S) + 128; }
constexpr int THREADS = 192;         // warps 0-3: epilogue (TMEM lanes), warp 4: producer, warp 5: MMA issue
constexpr uint32_t IDESC = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(CB >> 3) << 17) | ((uint32_t)(RB >> 4) << 24);
}  // namespace rki8

// 2^-e with 2^e > m (1 for m = 0).  A subnormal maximum would need 2^-e > 2^1023: the exponent is clamped there (the row is
// then sliced against a scale up to 2^51 too large: it keeps the bits above 2^-1078, i.e. all that a subnormal has).
// m = +Inf marks a row that holds a NaN or an Inf (rki8_rowmax_kernel): its scale is NaN, which the epilogue multiplies
// into every element of that row / column of S -- the FP64 tensor kernels propagate non-finite inputs the same way.
__device__ __forceinline__ double rki8_pow2_scale(double m) {
    if (!(m < __longlong_as_double(0x7ff0000000000000ll))) return __longlong_as_double(0x7ff8000000000000ll);
    return m > 0.0 ? scalbn(1.0, min(1023, -(ilogb(m) + 1))) : 1.0;
}

// Row maxima: mx[0][g] = max_p max(|Re|, |Im|) of Nb, mx[1 + iw][g] = max_p |w[iw][p]| max(|Re|, |Im|), as the bit patterns
// of non-negative doubles (ordered like unsigned integers: atomicMax).  mx must be zeroed before.
// grid (ceil(ng/128), p slices), block 128; the n_w <= MAXW running maxima of a thread live in registers.
constexpr int RKI8_MAXW = 32;
__global__ void __launch_bounds__(128) rki8_rowmax_kernel(const cd *__restrict__ Nb, int64_t ldn, int K, int ng,
                                                         const double *__restrict__ w, int64_t ldw, int n_w, int ngp,
                                                         unsigned long long *__restrict__ mx) {
    const int g = blockIdx.x * 128 + threadIdx.x;
    const int per = (K + gridDim.y - 1) / gridDim.y, p_lo = blockIdx.y * per, p_hi = min(K, p_lo + per);
    if (g >= ng) return;
    double m0 = 0.0, mw[RKI8_MAXW];
#pragma unroll
    for (int i = 0; i < RKI8_MAXW; i++) mw[i] = 0.0;
    for (int p = p_lo; p < p_hi; p++) {
        const cd v = Nb[(size_t)p * ldn + g];
        // fmax drops NaN operands: a NaN (or Inf) anywhere in the row must surface as a +Inf maximum instead
        const double inf = __longlong_as_double(0x7ff0000000000000ll);
        const double an = (v.x != v.x || v.y != v.y) ? inf : fmax(fabs(v.x), fabs(v.y));
        m0 = fmax(m0, an);
#pragma unroll
        for (int i = 0; i < RKI8_MAXW; i++)
            if (i < n_w) {
                const double t = fabs(w[(size_t)i * ldw + p]) * an;   // NaN weight, or 0 * Inf: NaN
                mw[i] = fmax(mw[i], t != t ? inf : t);
            }
    }
    atomicMax(&mx[g], (unsigned long long)__double_as_longlong(m0));
#pragma unroll
    for (int i = 0; i < RKI8_MAXW; i++)
        if (i < n_w) atomicMax(&mx[(size_t)(1 + i) * ngp + g], (unsigned long long)__double_as_longlong(mw[i]));
}
// inv[i] = 2^-e with 2^e > max, NaN for a non-finite row (in place over the bit patterns).  grid ceil(n/256), block 256.
__global__ void rki8_scale_finish_kernel(unsigned long long *__restrict__ mx, int n) {
    const int i = blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    const double m = __longlong_as_double((long long)mx[i]);
    reinterpret_cast<double *>(mx)[i] = rki8_pow2_scale(m);
}

// 16 values x (|x| < 1) -> S x 16 digit bytes, written as one 16-byte store per digit plane.  The value is rounded once to
// an integer v = rint(x 2^(6 + 7 (S - 1))) (|v| <= 2^48: exact in FP64 and in s64), and v is cut into balanced base-128
// digits from the least significant end with integer arithmetic: v = sum_i d_i 128^(S-1-i), d_i in [-64, 64].
template <int S>
__device__ __forceinline__ void rki8_store_digits(const double (&x)[16], int8_t *dst, int plane_stride) {
    uint32_t pk[S][4];
#pragma unroll
    for (int i = 0; i < S; i++)
#pragma unroll
        for (int q = 0; q < 4; q++) pk[i][q] = 0u;
    constexpr double SCALE = (double)(1ull << (6 + 7 * (S - 1)));
#pragma unroll
    for (int k = 0; k < 16; k++) {
        long long v = __double2ll_rn(x[k] * SCALE);
#pragma unroll
        for (int i = S - 1; i > 0; i--) {
            const long long d = ((v + 64) & 127) - 64;   // v mod 128 in [-64, 63]
            pk[i][k >> 2] |= ((uint32_t)d & 0xffu) << (8 * (k & 3));
            v = (v - d) >> 7;                            // exact: v - d is a multiple of 128
        }
        pk[0][k >> 2] |= ((uint32_t)v & 0xffu) << (8 * (k & 3));   // |v| <= 64
    }
#pragma unroll
    for (int i = 0; i < S; i++)
        *reinterpret_cast<uint4 *>(dst + (size_t)i * plane_stride) = make_uint4(pk[i][0], pk[i][1], pk[i][2], pk[i][3]);
}

// PL[rb][kb][digit][4096]: left rows R = rb 128 + r: half = R / ngp (0: [a | b], 1: [b | -a]), g = R % ngp (zero rows for
// g >= ng); K' column k' = kb 32 + kk: part = k' / Kpad, pair p = k' % Kpad.  grid (nkb, nrb), block 128.
template <int S>
__global__ void __launch_bounds__(128) rki8_pack_left_kernel(const cd *__restrict__ Nb, int64_t ldn, int Kpad, int ng, int ngp,
                                                            const double *__restrict__ invL, int8_t *__restrict__ PL) {
    const int kb = blockIdx.x, rb = blockIdx.y, r = threadIdx.x, nkb = gridDim.x;
    const int R = rb * rki8::RB + r, half = R / ngp, g = R - half * ngp;
    const int k0 = kb * rki8::KB, part = k0 / Kpad, p0 = k0 - part * Kpad;
    const bool valid = g < ng;
    const double sc = valid ? invL[g] : 0.0;
    // component: (half, part) = (0,0) a, (0,1) b, (1,0) b, (1,1) -a
    const bool take_im = (half ^ part) != 0;
    const double sgn = (half == 1 && part == 1) ? -sc : sc;
    int8_t *dst = PL + ((size_t)(rb * nkb + kb) * S) * rki8::A_BYTES + (r % 8) * 16 + (r / 8) * 256;
#pragma unroll
    for (int c = 0; c < 2; c++) {
        double x[16];
#pragma unroll
        for (int k = 0; k < 16; k++) {
            double v = 0.0;
            if (valid) {
                const cd z = Nb[(size_t)(p0 + c * 16 + k) * ldn + g];
                v = take_im ? z.y : z.x;
            }
            x[k] = v * sgn;
        }
        rki8_store_digits<S>(x, dst + c * 128, rki8::A_BYTES);
    }
}

// PR[iw][cb][kb][digit][2048]: rows g' = cb 64 + r, value w[iw][p] (a | b) 2^-eR.  The 32 components of a thread are read
// once and sliced for every frequency of the group.  grid (nkb, ncb), block 64.
template <int S>
__global__ void __launch_bounds__(64) rki8_pack_right_kernel(const cd *__restrict__ Nb, int64_t ldn, int Kpad, int ng, int ngp,
                                                            const double *__restrict__ w, int64_t ldw, int n_w,
                                                            const double *__restrict__ invR, int8_t *__restrict__ PR) {
    const int kb = blockIdx.x, cb = blockIdx.y, r = threadIdx.x, nkb = gridDim.x, ncb = gridDim.y;
    const int g = cb * rki8::CB + r;
    const int k0 = kb * rki8::KB, part = k0 / Kpad, p0 = k0 - part * Kpad;
    const bool valid = g < ng;
    double v[32];
#pragma unroll
    for (int k = 0; k < 32; k++) {
        v[k] = 0.0;
        if (valid) {
            const cd z = Nb[(size_t)(p0 + k) * ldn + g];
            v[k] = part ? z.y : z.x;
        }
    }
    for (int iw = 0; iw < n_w; iw++) {
        const double sc = valid ? invR[(size_t)iw * ngp + g] : 0.0;
        const double *wr = w + (size_t)iw * ldw + p0;
        int8_t *dst = PR + (((size_t)iw * ncb + cb) * nkb + kb) * S * rki8::B_BYTES + (r % 8) * 16 + (r / 8) * 256;
#pragma unroll
        for (int c = 0; c < 2; c++) {
            double x[16];
#pragma unroll
            for (int k = 0; k < 16; k++) x[k] = (v[c * 16 + k] * wr[c * 16 + k]) * sc;
            rki8_store_digits<S>(x, dst + c * 128, rki8::B_BYTES);
        }
    }
}

// One CTA = tile (rb, cb) of one frequency: tiles[] lists the tiles that meet the lower triangle.
// grid (n_tiles, n_w), block 192, dynamic shared memory rki8::smem_bytes(S).
// CL = 2: launched in clusters of two CTAs (consecutive blockIdx.x) whose tiles share the row block: each CTA fetches
// half of the row-block digits of a stage and multicasts it to both, so the L2 -> SM traffic of the row operand halves;
// a stage is released to the producers when the MMAs of BOTH CTAs have read it (multicast commit, barrier count 2).
template <int S, int CL>
__global__ void __launch_bounds__(rki8::THREADS, 1)
rank_k_i8_kernel(const int8_t *__restrict__ PL, const int8_t *__restrict__ PR, int nkb, int ncb, const int2 *__restrict__ tiles,
                 const double *__restrict__ invL, const double *__restrict__ invR, int ng, int ngp, cd *__restrict__ Sacc,
                 int64_t ldS, int64_t strideS) {
    using namespace rki8;
    constexpr int STAGE_BYTES = stage_bytes(S);
    static_assert(S * CB <= 512, "one TMEM accumulator of CB columns per digit level");
    extern __shared__ __align__(128) unsigned char i8_smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(i8_smem + STAGES * STAGE_BYTES);
    uint64_t *empty = full + STAGES;
    uint64_t *done = empty + STAGES;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(done + 1);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int2 tile = tiles[blockIdx.x];
    const int rb = tile.x, cb = tile.y, iw = blockIdx.y;
    uint32_t crank = 0;
    if constexpr (CL > 1) asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(crank));
    if (tid == 0) {
        for (int s = 0; s < STAGES; s++) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], CL);
        }
        mbar_init(done, 1);
        mbar_fence_init();
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(i8_saddr(tmem_slot)), "r"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if constexpr (CL > 1) {   // the peer's barriers must be initialised before anything is multicast to them
        asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t taddr = *tmem_slot;

    if (warp == 4) {
        if (lane == 0) {
            const int8_t *srcA = PL + (size_t)rb * nkb * S * A_BYTES;
            // a padding tile of an odd row (cb beyond the triangle) computes on the last column block and stores nothing
            const int8_t *srcB = PR + ((size_t)iw * ncb + min(cb, ncb - 1)) * nkb * S * B_BYTES;
            for (int kb = 0; kb < nkb; kb++) {
                const int s = kb % STAGES;
                if (kb >= STAGES) mbar_wait(&empty[s], ((kb / STAGES) - 1) & 1);
                unsigned char *st = i8_smem + s * STAGE_BYTES;
                mbar_arrive_expect_tx(&full[s], STAGE_BYTES);
                if constexpr (CL > 1) {
                    constexpr uint32_t PART = S * A_BYTES / CL;
                    static_assert(PART % 16 == 0, "bulk copies move multiples of 16 bytes");
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1], %2, [%3], %4;"
                                 ::"r"(smem_u32(st + crank * PART)), "l"(srcA + (size_t)kb * S * A_BYTES + crank * PART), "r"(PART),
                                   "r"(smem_u32(&full[s])), "h"((uint16_t)((1u << CL) - 1)) : "memory");
                } else {
                    bulk_g2s(st, srcA + (size_t)kb * S * A_BYTES, S * A_BYTES, &full[s]);
                }
                bulk_g2s(st + S * A_BYTES, srcB + (size_t)kb * S * B_BYTES, S * B_BYTES, &full[s]);
            }
        }
    } else if (warp == 5) {
        if (lane == 0) {
            for (int kb = 0; kb < nkb; kb++) {
                const int s = kb % STAGES;
                mbar_wait(&full[s], (kb / STAGES) & 1);
                asm volatile("tcgen05.fence::after_thread_sync;");
                const uint32_t sa = i8_saddr(i8_smem + s * STAGE_BYTES), sb = sa + S * A_BYTES;
                // Row digit i meets column digits j = 0 .. S-1-i; their planes are consecutive in shared memory (64 rows =
                // 8 core-matrix groups each) and their accumulators t = i + j are consecutive in TMEM, so up to 4 of them are
                // ONE MMA of N = 64 nj columns: the row operand is read 10 times per K block instead of 28 (S = 7), which
                // keeps the tensor core's shared-memory reads under 128 B/clk.
#pragma unroll
                for (int i = 0; i < S; i++) {
                    const uint64_t da = i8_smem_desc(sa + i * A_BYTES, 128, 256);
#pragma unroll
                    for (int j0 = 0; j0 + i < S; j0 += 4) {
                        const int nj = (S - i - j0) < 4 ? (S - i - j0) : 4;
                        const uint64_t db = i8_smem_desc(sb + j0 * B_BYTES, 128, 256);
                        const uint32_t idesc = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)((CB * nj) >> 3) << 17) | ((uint32_t)(RB >> 4) << 24);
                        // the first product into an accumulator is (kb, i) = (0, 0)
                        asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n}"
                                     ::"r"(taddr + (uint32_t)(i + j0) * CB), "l"(da), "l"(db), "r"(idesc), "r"((kb > 0 || i > 0) ? 1 : 0));
                    }
                }
                if constexpr (CL > 1) {   // arrive on the stage barrier of every CTA of the cluster
                    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                                 ::"r"(i8_saddr(&empty[s])), "h"((uint16_t)((1u << CL) - 1)) : "memory");
                } else {
                    i8_commit(&empty[s]);   // arrives when the MMAs above have read this stage
                }
            }
            i8_commit(done);
        }
    } else {
        // ---- epilogue: thread = TMEM lane = row of the tile ---------------------------------------------------------------
        mbar_wait(done, 0);
        asm volatile("tcgen05.fence::after_thread_sync;");
        const int R = rb * RB + tid, half = R / ngp, g = R - half * ngp;
        const bool row_ok = g < ng;
        const double sl = row_ok ? 1.0 / invL[g] : 0.0;
        cd *Srow = Sacc + (size_t)iw * strideS + (size_t)(row_ok ? g : 0) * ldS;
        const double *ir = invR + (size_t)iw * ngp;
        for (int c0 = 0; c0 < CB; c0 += 16) {
            double acc[16];
#pragma unroll
            for (int j = 0; j < 16; j++) acc[j] = 0.0;
            double f = 1.0;
#pragma unroll
            for (int t = 0; t < S; t++) {
                uint32_t r[16];
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                             : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                               "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                             : "r"(taddr + ((uint32_t)(warp * 32) << 16) + (uint32_t)(t * CB + c0)));
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                for (int j = 0; j < 16; j++) acc[j] = fma((double)(int32_t)r[j], f, acc[j]);
                f *= 0.0078125;   // 2^-7
            }
            if (row_ok) {
#pragma unroll
                for (int j = 0; j < 16; j++) {
                    const int gc = cb * CB + c0 + j;
                    if (gc <= g) {
                        const double v = acc[j] * sl * (1.0 / ir[gc]) * (1.0 / 4096.0);
                        cd *ptr = Srow + gc;
                        if (half == 0) ptr->x += v;
                        else ptr->y += v;
                    }
                }
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if constexpr (CL > 1) {   // no CTA leaves while its peer may still multicast into it or arrive on its barriers
        asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    }
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(512));
}
