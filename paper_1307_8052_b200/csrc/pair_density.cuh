// Pair densities on the |q+G| sphere (Table 1 steps 5-6; Eq. 7 / Eq. 12):
//   ntilde_nm(g) = (1/N) sum_j conj(u_n[j]) u_m[j] exp(-2 pi i (g1 j1/N1 + g2 j2/N2 + g3 j3/N3)),   g in the sphere.
//
// Two kernels, both pruned to the bounding box [g1min..g1max] x [g2min..g2max] x [g3min..g3max] of the sphere:
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
    cd *I;                          // [pair - p_begin][N1][ng2][ng3]
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

// Shared memory (all cd): tw3[N3] tw2[N2] | stage[2][2][RC*N3] (u_m, u_n chunks, double-buffered, filled by
// cp.async one chunk ahead) | zbuf[nbuf][RC*zpad(N3)] | Y0[N2*ng3] Y1[N2*ng3] ([row][g3i], g3i fastest).
__global__ void __launch_bounds__(256) pd_plane_kernel(const __grid_constant__ PdPlaneParams P) {
    extern __shared__ __align__(16) unsigned char pd_smem[];
    const int tid = threadIdx.x, nth = blockDim.x;
    const int N2 = P.N2, N3 = P.N3, ng2 = P.ng2, ng3 = P.ng3, RC = P.RC;
    const int N3p = zpad(N3) + 1;
    cd *tw3s = reinterpret_cast<cd *>(pd_smem);
    cd *tw2s = tw3s + N3;
    cd *stage = tw2s + N2;                        // [buf][um|un][RC*N3]
    cd *zbuf = stage + 4 * (size_t)RC * N3;       // [nbuf][RC*N3p]
    cd *Y0 = zbuf + (size_t)P.nbuf * RC * N3p;
    cd *Y1 = Y0 + (size_t)ng3 * N2;
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

    for (int q = 0; q < total; q++) {
        const int c = q % nchunks;
        const int row0 = c * RC;
        const int rc = min(RC, N2 - row0);
        cp_async_wait_all();
        __syncthreads();  // chunk q has landed; everybody is done with the buffers of chunk q-1
        if (q + 1 < total) prefetch(q + 1);

        // ---- z axis of chunk q -------------------------------------------------------------------------------
        const cd *sm = stage + (size_t)(q & 1) * 2 * RC * N3;
        const cd *sn = sm + (size_t)RC * N3;
        auto ld_g = [&](int line, int i) { return cmulc(sn[line * N3 + i], sm[line * N3 + i]); };
        auto st_y = [&](int line, int f, cd v) {
            const int gi = freq_to_box(f, N3, P.g3min, ng3);
            if (gi >= 0) Y0[(row0 + line) * ng3 + gi] = v;
        };
        if (P.pz.npass == 0) {
            for (int i = tid; i < rc; i += nth) Y0[(row0 + i) * ng3] = ld_g(i, 0);
        } else {
            int ns = 1;
            for (int ps = 0; ps < P.pz.npass; ps++) {
                const int R = P.pz.radix[ps];
                const bool first = (ps == 0), last = (ps == P.pz.npass - 1);
                const cd *s_ = zbuf + (size_t)((ps + 1) & 1) * RC * N3p;  // written by pass ps-1
                cd *d_ = zbuf + (size_t)(ps & 1) * RC * N3p;
                auto ld_s = [&](int line, int i) { return s_[line * N3p + zpad(i)]; };
                auto st_s = [&](int line, int i, cd v) { d_[line * N3p + zpad(i)] = v; };
                if (first && last) fft_pass_r<false>(R, tid, nth, rc, N3, ns, tw3s, ld_g, st_y);
                else if (first) fft_pass_r<false>(R, tid, nth, rc, N3, ns, tw3s, ld_g, st_s);
                else if (last) fft_pass_r<false>(R, tid, nth, rc, N3, ns, tw3s, ld_s, st_y);
                else fft_pass_r<false>(R, tid, nth, rc, N3, ns, tw3s, ld_s, st_s);
                ns *= R;
                if (!last) __syncthreads();
            }
        }
        if (c != nchunks - 1) continue;
        __syncthreads();

        // ---- last chunk of the pair: y axis on the ng3 surviving columns, then write out ---------------------------
        const int p = P.p_begin + blockIdx.y + (q / nchunks) * gridDim.y;
        cd *out;  // [g2i][g3i]
        if (P.py.npass == 0) {
            out = Y0;  // N2 == 1: Y0[0 * ng3 + g3i]
        } else {
            cd *src = Y0, *dst = Y1;
            int ns = 1;
            for (int ps = 0; ps < P.py.npass; ps++) {
                const int R = P.py.radix[ps];
                const bool last = (ps == P.py.npass - 1);
                cd *s_ = src, *d_ = dst;
                auto ld_s = [&](int line, int i) { return s_[i * ng3 + line]; };
                auto st_s = [&](int line, int i, cd v) { d_[i * ng3 + line] = v; };
                auto st_o = [&](int line, int f, cd v) {
                    const int gi = freq_to_box(f, N2, P.g2min, ng2);
                    if (gi >= 0) d_[gi * ng3 + line] = v;
                };
                if (last) fft_pass_r<true>(R, tid, nth, ng3, N2, ns, tw2s, ld_s, st_o);
                else fft_pass_r<true>(R, tid, nth, ng3, N2, ns, tw2s, ld_s, st_s);
                ns *= R;
                cd *t = src; src = dst; dst = t;
                __syncthreads();
            }
            out = src;
        }
        cd *Io = P.I + ((size_t)(p - P.p_begin) * P.N1 + j1) * nb2;
        for (int i = tid; i < nb2; i += nth) Io[i] = out[i];
        // the next pair's first z pass writes zbuf / Y0 only after the __syncthreads at the top of the loop
    }
}

// x axis + gather.  Thread (pair, b) with b = g2i*ng3 + g3i a column of the pruned box; tw1[t] = exp(-2 pi i t/N1).
// box2s[g1i*nb2 + b] = index of (g1min+g1i, ., .) in the sphere list, or -1 outside the sphere.
#define PD_G1_BLOCK 8
__global__ void __launch_bounds__(128) pd_xaxis_kernel(const cd *__restrict__ I, cd *__restrict__ Nbuf, int64_t ldn,
                                                      const cd *__restrict__ tw1, const int32_t *__restrict__ box2s,
                                                      int N1, int nb2, int g1min, int ng1, int p_begin, double inv_n) {
    extern __shared__ __align__(16) unsigned char pd_smem[];
    cd *tws = reinterpret_cast<cd *>(pd_smem);
    for (int i = threadIdx.x; i < N1; i += blockDim.x) tws[i] = tw1[i];
    __syncthreads();
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nb2) return;
    const int pl = blockIdx.y;
    const cd *Ip = I + (size_t)pl * N1 * nb2 + b;
    cd *out = Nbuf + (size_t)(p_begin + pl) * ldn;
    for (int gc = 0; gc < ng1; gc += PD_G1_BLOCK) {
        cd acc[PD_G1_BLOCK];
        int step[PD_G1_BLOCK], idx[PD_G1_BLOCK];
#pragma unroll
        for (int t = 0; t < PD_G1_BLOCK; t++) {
            acc[t] = cmake(0.0, 0.0);
            int g1 = g1min + gc + t;
            g1 %= N1;
            if (g1 < 0) g1 += N1;
            step[t] = g1;
            idx[t] = 0;
        }
        for (int j1 = 0; j1 < N1; j1++) {
            const cd x = Ip[(size_t)j1 * nb2];
#pragma unroll
            for (int t = 0; t < PD_G1_BLOCK; t++) {
                acc[t] = cfma(tws[idx[t]], x, acc[t]);
                idx[t] += step[t];
                if (idx[t] >= N1) idx[t] -= N1;
            }
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
