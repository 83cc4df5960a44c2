// Table 1 steps 3-4, upstream of the pair densities:
//   Eq. 10   u(r_j) = sum_Q C(Q) exp(+2 pi i (Q1 j1/N1 + Q2 j2/N2 + Q3 j3/N3))   plane waves -> grid
//   Eq. 11 u_out(r) = u_in(T^-1 r), conj under time reversal                      IBZ -> BZ
// The transform is separable and its INPUT is pruned (the coefficients fill a sphere inside the box
// [q1min..q1max] x [q2min..q2max] x [q3min..q3max]): x is expanded first on the box columns (nq1 terms per output,
// data still small), then one CTA per (band, x-plane) expands y on the nq3 box columns (nq2 terms) and z on all
// rows (nq3 terms) in shared memory and streams the plane out with coalesced 16-byte stores.  The work is per band,
// not per pair: for BASELINE.json configs[1] it is 1/12 of the pair-density traffic.
#pragma once
#include "common.cuh"

// T1[b][j1][c] = sum_q1i Cbox[q1i][c] exp(+2 pi i q1 j1 / N1); c = q2i nq3 + q3i a box column,
// table[q1i ncol + c] = index of that plane wave in C (or -1).  grid (ceil(ncol/128), N1, bands), block 128.
__global__ void __launch_bounds__(128) pw_xaxis_kernel(const cd *__restrict__ C, int n_pw, const int32_t *__restrict__ table,
                                                      const cd *__restrict__ tw1, int N1, int q1min, int nq1, int ncol,
                                                      cd *__restrict__ T1) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncol) return;
    const int j1 = blockIdx.y, b = blockIdx.z;
    const cd *Cb = C + (size_t)b * n_pw;
    cd acc = cmake(0.0, 0.0);
    int t = (int)(((int64_t)q1min * j1) % N1);
    if (t < 0) t += N1;
    for (int q = 0; q < nq1; q++) {
        const int idx = table[(size_t)q * ncol + c];
        if (idx >= 0) {
            const cd w = tw1[t];   // exp(-2 pi i t/N1); the inverse transform needs its conjugate
            acc = cfma(cmake(w.x, -w.y), Cb[idx], acc);
        }
        t += j1;
        if (t >= N1) t -= N1;
    }
    T1[((size_t)b * N1 + j1) * ncol + c] = acc;
}

// One CTA per (x-plane j1, band).  Shared memory (cd): tw2[N2] | tw3[N3] | P[nq2][nq3] | Y[N2][nq3].
//   Y[j2][q3i] = sum_q2i P[q2i][q3i] exp(+2 pi i q2 j2 / N2)
//   u[j2][j3]  = sum_q3i Y[j2][q3i] exp(+2 pi i q3 j3 / N3)      4 rows per thread share the twiddle
#define PW_ROWS 4
__global__ void __launch_bounds__(256) pw_zy_kernel(const cd *__restrict__ T1, const cd *__restrict__ tw2,
                                                   const cd *__restrict__ tw3, int N1, int N2, int N3, int q2min, int nq2,
                                                   int q3min, int nq3, cd *__restrict__ out) {
    extern __shared__ __align__(16) unsigned char pw_smem[];
    cd *tw2s = reinterpret_cast<cd *>(pw_smem);
    cd *tw3s = tw2s + N2;
    cd *P = tw3s + N3;
    cd *Y = P + (size_t)nq2 * nq3;
    const int tid = threadIdx.x, nth = blockDim.x;
    const int j1 = blockIdx.x, b = blockIdx.y;
    const int ncol = nq2 * nq3;
    for (int i = tid; i < N2; i += nth) tw2s[i] = tw2[i];
    for (int i = tid; i < N3; i += nth) tw3s[i] = tw3[i];
    const cd *Tp = T1 + ((size_t)b * N1 + j1) * ncol;
    for (int i = tid; i < ncol; i += nth) P[i] = Tp[i];
    __syncthreads();
    for (int i = tid; i < N2 * nq3; i += nth) {
        const int j2 = i / nq3, c3 = i - j2 * nq3;
        int t = (int)(((int64_t)q2min * j2) % N2);
        if (t < 0) t += N2;
        cd acc = cmake(0.0, 0.0);
        for (int q = 0; q < nq2; q++) {
            const cd w = tw2s[t];
            acc = cfma(cmake(w.x, -w.y), P[q * nq3 + c3], acc);
            t += j2;
            if (t >= N2) t -= N2;
        }
        Y[i] = acc;
    }
    __syncthreads();
    cd *op = out + ((size_t)b * N1 + j1) * N2 * N3;
    const int nrb = (N2 + PW_ROWS - 1) / PW_ROWS;
    for (int i = tid; i < nrb * N3; i += nth) {
        const int rb = i / N3, j3 = i - rb * N3;
        const int r0 = rb * PW_ROWS;
        int t = (int)(((int64_t)q3min * j3) % N3);
        if (t < 0) t += N3;
        cd acc[PW_ROWS];
#pragma unroll
        for (int r = 0; r < PW_ROWS; r++) acc[r] = cmake(0.0, 0.0);
        for (int q = 0; q < nq3; q++) {
            const cd w0 = tw3s[t];
            const cd w = cmake(w0.x, -w0.y);
#pragma unroll
            for (int r = 0; r < PW_ROWS; r++)
                if (r0 + r < N2) acc[r] = cfma(w, Y[(r0 + r) * nq3 + q], acc[r]);
            t += j3;
            if (t >= N3) t -= N3;
        }
#pragma unroll
        for (int r = 0; r < PW_ROWS; r++)
            if (r0 + r < N2) op[(size_t)(r0 + r) * N3 + j3] = acc[r];
    }
}

// out[b][j] = in[b][j'] (conjugated under time reversal), j'_i = sum_k S[i][k] j_k mod N_i with the integer matrix
// S[i][k] = M[i][k] N_i / N_k (M = T^-1 in reduced coordinates).  grid (ceil(N/256), bands).
struct RemapParams {
    int N1, N2, N3;
    int S[9];
    int conj;
};
__global__ void __launch_bounds__(256) symmetry_remap_kernel(const cd *__restrict__ in, cd *__restrict__ out,
                                                            const __grid_constant__ RemapParams R) {
    const int64_t N = (int64_t)R.N1 * R.N2 * R.N3;
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const int j3 = (int)(j % R.N3), j2 = (int)((j / R.N3) % R.N2), j1 = (int)(j / ((int64_t)R.N2 * R.N3));
    const int n[3] = {R.N1, R.N2, R.N3};
    int jp[3];
#pragma unroll
    for (int i = 0; i < 3; i++) {
        int64_t s = (int64_t)R.S[3 * i] * j1 + (int64_t)R.S[3 * i + 1] * j2 + (int64_t)R.S[3 * i + 2] * j3;
        s %= n[i];
        if (s < 0) s += n[i];
        jp[i] = (int)s;
    }
    cd v = in[(size_t)blockIdx.y * N + ((int64_t)jp[0] * R.N2 + jp[1]) * R.N3 + jp[2]];
    if (R.conj) v.y = -v.y;
    out[(size_t)blockIdx.y * N + j] = v;
}
