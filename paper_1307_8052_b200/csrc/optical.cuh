// Table 1 step 10: the optical limit q -> 0 of the G = 0 pair density.
//   Eq. 15 + Eq. 19  grad[al][n][m] = sum_Q conj(C_n(Q)) i (k + Q B)_al C_m(Q)
//                                                            + sum_a sum_ij conj(P^a_i,n) Qgrad^a_al[i][j] P^a_j,m
//   Eq. 13                       n_nm(G = 0) = -i qdir . grad[.][n][m] / (eps_m - eps_n)
// The gradient is taken in the plane-wave basis (the paper's FFT reformulation of the CPU code's 13-point stencil).
#pragma once
#include "common.cuh"

#define OPT_NB 4   // occupied bands per CTA

// grid (n_unocc, ceil(n_occ / OPT_NB)), block 128: threads stride over the plane waves, then a block reduction.
// Kc[al][q] = (k + Q_q B)_al (precomputed), C_occ [n_occ][n_pw], C_unocc [n_unocc][n_pw], grad [3][n_occ][n_unocc].
__global__ void __launch_bounds__(128) momentum_pw_kernel(const cd *__restrict__ C_occ, const cd *__restrict__ C_unocc,
                                                         const double *__restrict__ Kc, int n_pw, int n_occ, int n_unocc,
                                                         cd *__restrict__ grad) {
    __shared__ cd red[4][OPT_NB][3];
    const int m = blockIdx.x, n0 = blockIdx.y * OPT_NB;
    const cd *cm = C_unocc + (size_t)m * n_pw;
    cd acc[OPT_NB][3];
#pragma unroll
    for (int i = 0; i < OPT_NB; i++)
#pragma unroll
        for (int al = 0; al < 3; al++) acc[i][al] = cmake(0.0, 0.0);
    for (int q = threadIdx.x; q < n_pw; q += blockDim.x) {
        const cd c = cm[q];
        const double k0 = Kc[q], k1 = Kc[n_pw + q], k2 = Kc[2 * (size_t)n_pw + q];
#pragma unroll
        for (int i = 0; i < OPT_NB; i++) {
            if (n0 + i < n_occ) {
                const cd t = cmulc(C_occ[(size_t)(n0 + i) * n_pw + q], c);   // conj(C_n) C_m
                acc[i][0] = cfma(cmake(k0, 0.0), t, acc[i][0]);
                acc[i][1] = cfma(cmake(k1, 0.0), t, acc[i][1]);
                acc[i][2] = cfma(cmake(k2, 0.0), t, acc[i][2]);
            }
        }
    }
    // fixed-order reduction: lanes by shuffles, then the 4 warps through shared memory
#pragma unroll
    for (int i = 0; i < OPT_NB; i++)
#pragma unroll
        for (int al = 0; al < 3; al++) {
            cd v = acc[i][al];
            for (int o = 16; o > 0; o >>= 1) {
                v.x += __shfl_down_sync(0xffffffffu, v.x, o);
                v.y += __shfl_down_sync(0xffffffffu, v.y, o);
            }
            if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5][i][al] = v;
        }
    __syncthreads();
    if (threadIdx.x < OPT_NB * 3) {
        const int i = threadIdx.x / 3, al = threadIdx.x % 3;
        if (n0 + i < n_occ) {
            cd s = red[0][i][al];
            for (int wv = 1; wv < 4; wv++) s = cadd(s, red[wv][i][al]);
            grad[((size_t)al * n_occ + n0 + i) * n_unocc + m] = mul_pos_i(s);   // the factor i of i (k + Q)
        }
    }
}

// grad[al][n][m] += sum_a sum_ij conj(P_occ[n][poff_a + i]) Qgrad[a][al][i][j] P_unocc[m][poff_a + j]
// grid (ceil(n_unocc / 128), n_occ, 3), block 128.
__global__ void __launch_bounds__(128) momentum_paw_kernel(cd *__restrict__ grad, int n_occ, int n_unocc, int ptot, int n_atoms,
                                                          const int *__restrict__ atom_poff, const int *__restrict__ atom_ni,
                                                          const cd *__restrict__ P_occ, const cd *__restrict__ P_unocc,
                                                          const cd *__restrict__ Qgrad) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x, n = blockIdx.y, al = blockIdx.z;
    if (m >= n_unocc) return;
    cd acc = cmake(0.0, 0.0);
    size_t qoff = 0;
    for (int a = 0; a < n_atoms; a++) {
        const int ni = atom_ni[a], po = atom_poff[a];
        const cd *Qa = Qgrad + qoff + (size_t)al * ni * ni;
        for (int i = 0; i < ni; i++) {
            cd row = cmake(0.0, 0.0);
            for (int j = 0; j < ni; j++) row = cfma(Qa[i * ni + j], P_unocc[(size_t)m * ptot + po + j], row);
            acc = cadd(acc, cmulc(P_occ[(size_t)n * ptot + po + i], row));
        }
        qoff += (size_t)3 * ni * ni;
    }
    cd *o = grad + ((size_t)al * n_occ + n) * n_unocc + m;
    *o = cadd(*o, acc);
}

// N[p][idx0] = -i (qdir . grad[.][n][m]) / (eps_m - eps_n) for the pairs p of a batch (n = n0 + p / mlen, m = m0 + p % mlen).
__global__ void optical_head_kernel(cd *__restrict__ Nbuf, int64_t ldn, int idx0, int K, int n0, int mlen, int m0, int n_occ,
                                    int n_unocc, const double *__restrict__ eps_occ, const double *__restrict__ eps_unocc,
                                    double q0, double q1, double q2, const cd *__restrict__ grad) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= K) return;
    const int n = n0 + p / mlen, m = m0 + p % mlen;
    const size_t plane = (size_t)n_occ * n_unocc, at = (size_t)n * n_unocc + m;
    const cd g0 = grad[at], g1 = grad[plane + at], g2 = grad[2 * plane + at];
    const cd s = cmake(q0 * g0.x + q1 * g1.x + q2 * g2.x, q0 * g0.y + q1 * g1.y + q2 * g2.y);
    const double de = eps_unocc[m] - eps_occ[n];
    Nbuf[(size_t)p * ldn + idx0] = de != 0.0 ? cscale(1.0 / de, mul_neg_i(s)) : cmake(0.0, 0.0);
}
