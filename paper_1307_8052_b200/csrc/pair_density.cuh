// Pair densities on the |q+G| sphere (Table 1 steps 5-6; Eq. 7 / Eq. 12):
//   ntilde_nm(g) = (1/N) sum_j conj(u_n[j]) u_m[j] exp(-2 pi i (g1 j1/N1 + g2 j2/N2 + g3 j3/N3)),   g in the sphere.
//
// The general path (any plane whose lengths factor into 2, 3, 5, 7; pd_zy_kernel of pair_density_zy.cuh replaces the
// first kernel for the plane shapes it is specialised for).  Two kernels, both pruned to the bounding box [g1min..g1max] x [g2min..g2max] x [g3min..g3max] of the sphere:
//   pd_plane_kernel  one CTA per (x-plane j1, pair): the plane u[j1][:][:] is contiguous in HBM (N2*N3*16 B), so it
//                    is streamed once with fully coalesced 16-byte loads; the product conj(u_n) u_m is formed in
//                    registers on the way into the first radix pass of the z FFT; z lines are transformed in
//                    shared memory, only the ng3 needed frequencies survive; then the y FFT runs on those ng3
//                    columns and only ng2 frequencies survive.  Output I[pair][j1][g2i][g3i] is 5-10 % of the
//                    input volume and stays in L2 for the second kernel.
//   pd_xaxis_kernel  the x transform restricted to ng1 frequencies is a (ng1 x N1) DFT matrix applied to the
//                    pruned data (direct sum; cheaper than an FFT once ng1 << N1), scaled by 1/N and scattered
//                    to the sphere order of the N buffer (the gather of step 6).
#pragma once
#include "fft.cuh"

struct PdPlaneParams {
    const cd *psi_occ, *psi_unocc;  // [band][N1][N2][N3]
    cd *I;                          // [pair - p_begin][N1][ncols]: only the (g2, g3) columns that hold sphere points
    const int32_t *coltab;          // [ncols]: (g2i << 16) | g3i of column c
    int ncols;
    const cd *tw3, *tw2;            // exp(-2 pi i t/N3), exp(-2 pi i t/N2)
    int N1, N2, N3;
    int n0, mlen, m0;               // pair p of the batch -> band n = n0 + p / mlen, m = m0 + p % mlen
    int p_begin, p_count;           // pairs of the batch handled by this launch
    int g2min, ng2, g3min, ng3;
    int RC;                         // z lines per chunk
    int nbuf;                       // z ping-pong buffers in shared memory (0, 1 or 2)
    FftPlan pz, py;
};

__device__ __forceinline__ int freq_to_box(int f, int n, int gmin, int ngb) {
    const int g = (2 * f < n) ? f : f - n;
    const int i = g - gmin;
    return (i >= 0 && i < ngb) ? i : -1;
}

// element index -> padded index inside a z line: one spare slot per 8 elements turns the stride-R stores of the
// first Stockham pass (R = 4, 8: 64 / 128-byte strides) into conflict-free ones.
__device__ __forceinline__ int zpad(int i) { return i + (i >> 3); }

__device__ __forceinline__ void cp_async16(void *dst_smem, const void *src_gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// Compile-time pass chains for grid lengths known when the library is built (the radices, butterfly counts and
// index arithmetic then fold into constants); the run-time loops below them serve every other length.
template <int NC, int PS, int NS, class LDG, class STY, class MKLD, class MKST>
__device__ __forceinline__ void z_passes_ct(int tid, int nth, int rc, const cd *tw, LDG ld_g, STY st_y, MKLD mk_ld,
                                            MKST mk_st) {
    constexpr FftPlanResult pr = fft_plan_c(NC);
    if constexpr (PS < pr.plan.npass) {
        constexpr int R = pr.plan.radix[PS];
        constexpr bool first = (PS == 0), last = (PS == pr.plan.npass - 1);
        auto ld_s = mk_ld(PS);
        auto st_s = mk_st(PS);
        if constexpr (first && last) fft_pass<R, false, NC, NS>(tid, nth, rc, NC, NS, tw, ld_g, st_y);
        else if constexpr (first) fft_pass<R, false, NC, NS>(tid, nth, rc, NC, NS, tw, ld_g, st_s);
        else if constexpr (last) fft_pass<R, false, NC, NS>(tid, nth, rc, NC, NS, tw, ld_s, st_y);
        else fft_pass<R, false, NC, NS>(tid, nth, rc, NC, NS, tw, ld_s, st_s);
        if constexpr (!last) {
            __syncthreads();
            z_passes_ct<NC, PS + 1, NS * R>(tid, nth, rc, tw, ld_g, st_y, mk_ld, mk_st);
        }
    }
}

template <int NC, int PS, int NS, class MKLD, class MKST, class MKSTO>
__device__ __forceinline__ void y_passes_ct(int tid, int nth, int nlines, const cd *tw, MKLD mk_ld, MKST mk_st,
                                            MKSTO mk_sto) {
    constexpr FftPlanResult pr = fft_plan_c(NC);
    if constexpr (PS < pr.plan.npass) {
        constexpr int R = pr.plan.radix[PS];
        constexpr bool last = (PS == pr.plan.npass - 1);
        auto ld_s = mk_ld(PS);
        if constexpr (last) fft_pass<R, true, NC, NS>(tid, nth, nlines, NC, NS, tw, ld_s, mk_sto(PS));
        else fft_pass<R, true, NC, NS>(tid, nth, nlines, NC, NS, tw, ld_s, mk_st(PS));
        __syncthreads();
        y_passes_ct<NC, PS + 1, NS * R>(tid, nth, nlines, tw, mk_ld, mk_st, mk_sto);
    }
}

// Shared memory (all cd): tw3[N3] tw2[N2] | stage[2][2][RC*N3] (u_m, u_n chunks, double-buffered, filled by
// cp.async one chunk ahead) | zbuf[nbuf][RC*zpad(N3)] | Y[2][N2*ng3] ([row][g3i], g3i fastest).
// N3C, N2C > 0: grid lengths fixed at compile time (must equal P.N3, P.N2); 0: run-time lengths.
template <int N3C, int N2C>
__global__ void __launch_bounds__(256) pd_plane_kernel(const __grid_constant__ PdPlaneParams P) {
    extern __shared__ __align__(16) unsigned char pd_smem[];
    const int tid = threadIdx.x, nth = blockDim.x;
    const int N2 = N2C > 0 ? N2C : P.N2, N3 = N3C > 0 ? N3C : P.N3;
    const int ng2 = P.ng2, ng3 = P.ng3, RC = P.RC;
    const int N3p = zpad(N3) + 1;
    cd *tw3s = reinterpret_cast<cd *>(pd_smem);
    cd *tw2s = tw3s + N3;
    cd *stage = tw2s + N2;                        // [buf][um|un][RC*N3]
    cd *zbuf = stage + 4 * (size_t)RC * N3;       // [nbuf][RC*N3p]
    cd *Y = zbuf + (size_t)P.nbuf * RC * N3p;     // [2][N2*ng3]
    const int ysz = ng3 * N2;
    for (int i = tid; i < N3; i += nth) tw3s[i] = P.tw3[i];
    for (int i = tid; i < N2; i += nth) tw2s[i] = P.tw2[i];

    const int j1 = blockIdx.x;
    const size_t plane = (size_t)N2 * N3;
    const size_t vol = plane * P.N1;
    const int nb2 = ng2 * ng3;
    const int nchunks = (N2 + RC - 1) / RC;
    const int npairs = (P.p_count - (int)blockIdx.y + (int)gridDim.y - 1) / (int)gridDim.y;  // pairs of this CTA
    const int total = npairs * nchunks;

    // chunk q of this CTA: pair p = p_begin + blockIdx.y + (q / nchunks) * gridDim.y, rows [c*RC, c*RC + rc)
    auto prefetch = [&](int q) {
        const int p = P.p_begin + blockIdx.y + (q / nchunks) * gridDim.y;
        const int row0 = (q % nchunks) * RC;
        const int cnt = min(RC, N2 - row0) * N3;
        const int n = P.n0 + p / P.mlen, m = P.m0 + p % P.mlen;
        const cd *um = P.psi_unocc + (size_t)m * vol + (size_t)j1 * plane + (size_t)row0 * N3;
        const cd *un = P.psi_occ + (size_t)n * vol + (size_t)j1 * plane + (size_t)row0 * N3;
        cd *sm = stage + (size_t)(q & 1) * 2 * RC * N3;
        cd *sn = sm + (size_t)RC * N3;
        for (int i = tid; i < cnt; i += nth) {
            cp_async16(sm + i, um + i);
            cp_async16(sn + i, un + i);
        }
        cp_async_commit();
    };
    if (total > 0) prefetch(0);

    int c = 0, pi = 0;  // chunk within the pair, pair counter of this CTA
    for (int q = 0; q < total; q++) {
        const int row0 = c * RC;
        const int rc = min(RC, N2 - row0);
        cp_async_wait_all();
        __syncthreads();  // chunk q has landed; everybody is done with the buffers of chunk q-1
        if (q + 1 < total) prefetch(q + 1);

        // ---- z axis of chunk q -------------------------------------------------------------------------------
        const cd *sm = stage + (size_t)(q & 1) * 2 * RC * N3;
        const cd *sn = sm + (size_t)RC * N3;
        cd *Y0 = Y;
        auto ld_g = [=](int line, int i) { return cmulc(sn[line * N3 + i], sm[line * N3 + i]); };
        auto st_y = [=](int line, int f, cd v) {
            const int gi = freq_to_box(f, N3, P.g3min, ng3);
            if (gi >= 0) Y0[(row0 + line) * ng3 + gi] = v;
        };
        auto mk_ld = [=](int ps) {
            const cd *s_ = zbuf + (size_t)((ps + 1) & 1) * RC * N3p;  // written by pass ps-1
            return [=](int line, int i) { return s_[line * N3p + zpad(i)]; };
        };
        auto mk_st = [=](int ps) {
            cd *d_ = zbuf + (size_t)(ps & 1) * RC * N3p;
            return [=](int line, int i, cd v) { d_[line * N3p + zpad(i)] = v; };
        };
        if constexpr (N3C > 0) {
            z_passes_ct<N3C, 0, 1>(tid, nth, rc, tw3s, ld_g, st_y, mk_ld, mk_st);
        } else if (P.pz.npass == 0) {
            for (int i = tid; i < rc; i += nth) Y0[(row0 + i) * ng3] = ld_g(i, 0);
        } else {
            int ns = 1;
            for (int ps = 0; ps < P.pz.npass; ps++) {
                const int R = P.pz.radix[ps];
                const bool first = (ps == 0), last = (ps == P.pz.npass - 1);
                auto ld_s = mk_ld(ps);
                auto st_s = mk_st(ps);
                if (first && last) fft_pass_r<false>(R, tid, nth, rc, N3, ns, tw3s, ld_g, st_y);
                else if (first) fft_pass_r<false>(R, tid, nth, rc, N3, ns, tw3s, ld_g, st_s);
                else if (last) fft_pass_r<false>(R, tid, nth, rc, N3, ns, tw3s, ld_s, st_y);
                else fft_pass_r<false>(R, tid, nth, rc, N3, ns, tw3s, ld_s, st_s);
                ns *= R;
                if (!last) __syncthreads();
            }
        }
        if (++c < nchunks) continue;
        c = 0;
        __syncthreads();

        // ---- last chunk of the pair: y axis on the ng3 surviving columns, then write out ---------------------------
        const int p = P.p_begin + blockIdx.y + pi * gridDim.y;
        pi++;
        // pass ps reads Y[ps & 1] and writes Y[(ps + 1) & 1]; the last pass writes [g2i][g3i]
        auto my_ld = [=](int ps) {
            const cd *s_ = Y + (size_t)(ps & 1) * ysz;
            return [=](int line, int i) { return s_[i * ng3 + line]; };
        };
        auto my_st = [=](int ps) {
            cd *d_ = Y + (size_t)((ps + 1) & 1) * ysz;
            return [=](int line, int i, cd v) { d_[i * ng3 + line] = v; };
        };
        auto my_sto = [=](int ps) {
            cd *d_ = Y + (size_t)((ps + 1) & 1) * ysz;
            return [=](int line, int f, cd v) {
                const int gi = freq_to_box(f, N2, P.g2min, ng2);
                if (gi >= 0) d_[gi * ng3 + line] = v;
            };
        };
        int npy;
        if constexpr (N2C > 0) {
            constexpr FftPlanResult pr = fft_plan_c(N2C);
            npy = pr.plan.npass;
            y_passes_ct<N2C, 0, 1>(tid, nth, ng3, tw2s, my_ld, my_st, my_sto);
        } else {
            npy = P.py.npass;  // 0 when N2 == 1: Y[0][0 * ng3 + g3i] is already [g2i = 0][g3i]
            int ns = 1;
            for (int ps = 0; ps < npy; ps++) {
                const int R = P.py.radix[ps];
                if (ps == npy - 1) fft_pass_r<true>(R, tid, nth, ng3, N2, ns, tw2s, my_ld(ps), my_sto(ps));
                else fft_pass_r<true>(R, tid, nth, ng3, N2, ns, tw2s, my_ld(ps), my_st(ps));
                ns *= R;
                __syncthreads();
            }
        }
        const cd *out = Y + (size_t)(npy & 1) * ysz;
        cd *Io = P.I + ((size_t)(p - P.p_begin) * P.N1 + j1) * P.ncols;   // only the columns that hold sphere points
        for (int i = tid; i < P.ncols; i += nth) {
            const int oc = P.coltab[i];
            Io[i] = out[(oc >> 16) * ng3 + (oc & 0xffff)];
        }
        // the next pair's first z pass writes zbuf / Y only after the __syncthreads at the top of the loop
    }
}

typedef void (*PdPlaneKernel)(const PdPlaneParams);

// x axis + gather.  Thread (pair, b) with b = g2i*ng3 + g3i a column of the pruned box; tw1[t] = exp(-2 pi i t/N1).
// box2s[g1i*nb2 + b] = index of (g1min+g1i, column b) in the sphere list, or -1 outside the sphere; nb2 = kept (g2, g3) columns.
// The (ng1 x N1) DFT matrix of the kept frequencies is tabulated in shared memory ([j1][g1i], read as a warp-wide
// broadcast); a thread keeps PD_G1_BLOCK accumulators, so a sphere with ng1 <= PD_G1_BLOCK reads I once, and the
// loads of four x planes are issued together to cover the L2 latency.
// Dynamic shared memory: N1 * PD_G1_BLOCK * sizeof(cd).
// Row of the N buffer that pair pl of a launch goes to.  A plain launch covers the batch's pairs p_begin, p_begin + 1, ...
// (win.len = INT_MAX: row = p_begin + pl).  A window launch (streamed k-point: some unoccupied bands of every occupied row)
// numbers its pairs row by row over the window, p' = p_begin + pl = r win.len + j, and they belong to the batch's rows
// r win.stride + win.off + j.
struct PdRowWindow {
    int len, stride, off;
};
__device__ __forceinline__ size_t pd_out_row(int p, PdRowWindow win) {
    const int r = p / win.len;
    return (size_t)r * win.stride + win.off + (p - r * win.len);
}
#define PD_G1_BLOCK 16
__global__ void __launch_bounds__(128) pd_xaxis_kernel(const cd *__restrict__ I, cd *__restrict__ Nbuf, int64_t ldn,
                                                      const cd *__restrict__ tw1, const int32_t *__restrict__ box2s,
                                                      int N1, int nb2, int g1min, int ng1, int p_begin, double inv_n, PdRowWindow win) {
    extern __shared__ __align__(16) unsigned char pd_smem[];
    cd *twt = reinterpret_cast<cd *>(pd_smem);   // [j1][t]
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    const bool act = b < nb2;
    const int pl = blockIdx.y;
    const cd *Ip = I + (size_t)pl * N1 * nb2 + (act ? b : 0);
    cd *out = Nbuf + pd_out_row(p_begin + pl, win) * ldn;
    for (int gc = 0; gc < ng1; gc += PD_G1_BLOCK) {
        __syncthreads();
        for (int i = threadIdx.x; i < N1 * PD_G1_BLOCK; i += blockDim.x) {
            const int j1 = i / PD_G1_BLOCK, t = i - j1 * PD_G1_BLOCK;
            int g1 = (g1min + gc + t) % N1;
            if (g1 < 0) g1 += N1;
            twt[i] = (gc + t < ng1) ? tw1[(int)(((int64_t)g1 * j1) % N1)] : cmake(0.0, 0.0);
        }
        __syncthreads();
        cd acc[PD_G1_BLOCK];
#pragma unroll
        for (int t = 0; t < PD_G1_BLOCK; t++) acc[t] = cmake(0.0, 0.0);
        if (act) {
            int j1 = 0;
            for (; j1 + 4 <= N1; j1 += 4) {
                cd x[4];
#pragma unroll
                for (int u = 0; u < 4; u++) x[u] = Ip[(size_t)(j1 + u) * nb2];
#pragma unroll
                for (int u = 0; u < 4; u++)
#pragma unroll
                    for (int t = 0; t < PD_G1_BLOCK; t++) acc[t] = cfma(twt[(j1 + u) * PD_G1_BLOCK + t], x[u], acc[t]);
            }
            for (; j1 < N1; j1++) {
                const cd x = Ip[(size_t)j1 * nb2];
#pragma unroll
                for (int t = 0; t < PD_G1_BLOCK; t++) acc[t] = cfma(twt[j1 * PD_G1_BLOCK + t], x, acc[t]);
            }
#pragma unroll
            for (int t = 0; t < PD_G1_BLOCK; t++) {
                if (gc + t < ng1) {
                    const int s = box2s[(size_t)(gc + t) * nb2 + b];
                    if (s >= 0) out[s] = cscale(inv_n, acc[t]);
                }
            }
        }
    }
}

// x axis + gather with the two-level split N1 = 8 NB (N1 % 8 == 0, at most PD_X8_ND_MAX kept frequencies per residue mod 8):
//   A_j[k1] = sum_s x[j + NB s] W_8^(s k1)   (radix-8 butterfly over 8 planes loaded together),
//   X[f]    = sum_j W_N1^(j f) A_j[f mod 8]  for the ng1 kept f = k1 + 8 d only:
// 8 independent loads in flight per thread and NB (8 log 8 + ng1) instead of N1 ng1 multiply-adds per column.
// Dynamic shared memory: N1 * PD_X8_ND * sizeof(cd) (twiddle products per (j, kept-frequency slot)).  Same arguments
// as pd_xaxis_kernel.
#define PD_X8_ND_MAX 3
// NBT > 0: N1 = 8 NBT known at compile time (short x axes: the 24^3 and 16^3 grids): the j loop is unrolled, so all 8 NBT
// loads of a column are in flight together.  grid (ceil(nb2 / 128), pairs handled concurrently): a block walks over the
// pairs pl = blockIdx.y, blockIdx.y + gridDim.y, ... of the launch, so the twiddle table, the kept-slot mask and the
// column's scatter indices are set up once per block and not once per pair.
template <int PD_X8_ND, int NBT>   // PD_X8_ND: kept-frequency slots per residue mod 8 (2 when the box needs no more: fewer registers)
__global__ void __launch_bounds__(128, 4) pd_xaxis8_kernel(const cd *__restrict__ I, cd *__restrict__ Nbuf, int64_t ldn,
                                                       const cd *__restrict__ tw1, const int32_t *__restrict__ box2s,
                                                       int N1, int nb2, int g1min, int ng1, int p_begin, int p_count, double inv_n, PdRowWindow win) {
    extern __shared__ __align__(16) unsigned char pd_smem[];
    cd *twt = reinterpret_cast<cd *>(pd_smem);   // [j][slot], slot = k1 PD_X8_ND + d: W_N1^(j f_slot)
    const int NB = NBT > 0 ? NBT : (N1 >> 3);
    // kept frequencies of residue k1: f = k1 + 8 (dlo + d), box index f - g1min (the same for every thread)
    const int dlo = (g1min >= 0 ? g1min : g1min - 7) / 8;
    for (int i = threadIdx.x; i < NB * 8 * PD_X8_ND; i += blockDim.x) {
        const int j = i / (8 * PD_X8_ND), slot = i - j * 8 * PD_X8_ND;
        const int f = slot / PD_X8_ND + 8 * (dlo + slot % PD_X8_ND);
        int fp = f % N1;
        if (fp < 0) fp += N1;
        twt[i] = tw1[(int)(((int64_t)fp * j) % N1)];
    }
    uint32_t mask = 0;
#pragma unroll
    for (int slot = 0; slot < 8 * PD_X8_ND; slot++) {
        const int gi = slot / PD_X8_ND + 8 * (dlo + slot % PD_X8_ND) - g1min;
        if (gi >= 0 && gi < ng1) mask |= 1u << slot;
    }
    __syncthreads();
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nb2) return;
    // short axes: the sphere index of every kept slot of this column (-1: outside the sphere) is the same for all pairs
    int sidx[NBT > 0 ? 8 : 1][PD_X8_ND];
    if constexpr (NBT > 0) {
#pragma unroll
        for (int k1 = 0; k1 < 8; k1++)
#pragma unroll
            for (int d = 0; d < PD_X8_ND; d++) {
                sidx[k1][d] = -1;
                if (mask & (1u << (k1 * PD_X8_ND + d))) sidx[k1][d] = box2s[(size_t)(k1 + 8 * (dlo + d) - g1min) * nb2 + b];
            }
    }
    for (int pl = blockIdx.y; pl < p_count; pl += gridDim.y) {
        const cd *Ip = I + (size_t)pl * N1 * nb2 + b;
        cd acc[8][PD_X8_ND];
#pragma unroll
        for (int k1 = 0; k1 < 8; k1++)
#pragma unroll
            for (int d = 0; d < PD_X8_ND; d++) acc[k1][d] = cmake(0.0, 0.0);
        auto body = [&](int j) {
            cd v[8];
#pragma unroll
            for (int s = 0; s < 8; s++) v[s] = Ip[(size_t)(j + NB * s) * nb2];
            Bfly<8>::run(v);
            const cd *tj = twt + j * 8 * PD_X8_ND;
#pragma unroll
            for (int k1 = 0; k1 < 8; k1++)
#pragma unroll
                for (int d = 0; d < PD_X8_ND; d++)
                    if (mask & (1u << (k1 * PD_X8_ND + d))) acc[k1][d] = cfma(tj[k1 * PD_X8_ND + d], v[k1], acc[k1][d]);
        };
        if constexpr (NBT > 0) {
#pragma unroll
            for (int j = 0; j < NBT; j++) body(j);
        } else {
#pragma unroll 1
            for (int j = 0; j < NB; j++) body(j);
        }
        cd *out = Nbuf + pd_out_row(p_begin + pl, win) * ldn;
#pragma unroll
        for (int k1 = 0; k1 < 8; k1++)
#pragma unroll
            for (int d = 0; d < PD_X8_ND; d++) {
                if constexpr (NBT > 0) {
                    if (sidx[k1][d] >= 0) out[sidx[k1][d]] = cscale(inv_n, acc[k1][d]);
                } else if (mask & (1u << (k1 * PD_X8_ND + d))) {
                    const int s = box2s[(size_t)(k1 + 8 * (dlo + d) - g1min) * nb2 + b];
                    if (s >= 0) out[s] = cscale(inv_n, acc[k1][d]);
                }
            }
    }
}
// can pd_xaxis8_kernel serve this x axis?  (every kept frequency must fall in one of its PD_X8_ND slots per residue)
// returns the number of slots needed (2 or 3), or 0 if the kernel cannot serve this x axis
static inline int pd_xaxis8_slots(int N1, int g1min, int ng1) {
    if (N1 % 8 != 0 || N1 < 16 || ng1 > N1) return 0;
    const int dlo = (g1min >= 0 ? g1min : g1min - 7) / 8;
    const int gmax = g1min + ng1 - 1;
    const int dhi = (gmax >= 0 ? gmax : gmax - 7) / 8;
    const int nd = dhi - dlo + 1;
    if (nd > PD_X8_ND_MAX || 8 * nd > N1) return 0;
    return nd <= 2 ? 2 : 3;
}
