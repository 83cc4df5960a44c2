// Table 1 steps 3-4, upstream of the pair densities:
//   Eq. 10   u(r_j) = sum_Q C(Q) exp(+2 pi i (Q1 j1/N1 + Q2 j2/N2 + Q3 j3/N3))   plane waves -> grid
//   Eq. 11 u_out(r) = u_in(T^-1 r), conj under time reversal                      IBZ -> BZ
// The transform is separable and its INPUT is pruned (the coefficients fill a sphere inside the box
// [q1min..q1max] x [q2min..q2max] x [q3min..q3max]): x is expanded first on the box columns (nq1 terms per output,
// data still small), then one CTA per (band, x-plane) expands y on the nq3 box columns (nq2 terms) and z on all
// rows (nq3 terms) in shared memory and streams the plane out with coalesced 16-byte stores.  The work is per band,
// not per pair: for BASELINE.json configs[1] it is 1/12 of the pair-density traffic.
#pragma once
#include "fft.cuh"

// Input-pruned inverse transform of one line by the two-level split N = NA NB (the transpose of the forward
// pair-density split): for the outputs j + NB s (s < NA) of one j < NB,
//   Z[k1] = sum_{q in box, q = k1 mod NA} x[q] exp(+2 pi i q j / N),      u[j + NB s] = sum_k1 exp(+2 pi i k1 s / NA) Z[k1],
// i.e. nq twiddled terms per j (not per output) followed by one inverse radix-NA butterfly in registers
// (inverse = conj o forward o conj).  NA = 1 degenerates to the direct sum.
//   ld(qi) reads x at box position qi (q = qmin + qi), st(n, v) writes output n.
template <int NA, class LD, class ST>
__device__ __forceinline__ void pw_expand_line(int N, int j, int qmin, int nq, const cd *__restrict__ tw, LD ld, ST st) {
    const int NB = N / NA;
    int r0 = qmin % NA;
    if (r0 < 0) r0 += NA;                              // the box is read from q0 = qmin - r0 = 0 (mod NA): k1 = position mod NA
    const int q0 = qmin - r0;
    const int step = (int)(((int64_t)NA * j) % N);     // twiddle index step between q and q + NA
    cd z[NA];
    int t[NA];
#pragma unroll
    for (int k1 = 0; k1 < NA; k1++) {
        z[k1] = cmake(0.0, 0.0);
        int tt = (int)(((int64_t)(q0 + k1) * j) % N);
        t[k1] = tt < 0 ? tt + N : tt;
    }
    for (int base = -r0; base < nq; base += NA) {      // NA independent accumulations per trip
#pragma unroll
        for (int k1 = 0; k1 < NA; k1++) {
            const int qi = base + k1;
            if (qi >= 0 && qi < nq) {
                const cd w = tw[t[k1]];                // exp(-2 pi i t/N): the inverse needs the conjugate
                z[k1] = cfma(cmake(w.x, -w.y), ld(qi), z[k1]);
            }
            t[k1] += step;
            if (t[k1] >= N) t[k1] -= N;
        }
    }
    if constexpr (NA > 1) {                            // inverse butterfly = conj o forward o conj
#pragma unroll
        for (int k1 = 0; k1 < NA; k1++) z[k1].y = -z[k1].y;
        Bfly<NA>::run(z);
#pragma unroll
        for (int s = 0; s < NA; s++) z[s].y = -z[s].y;
    }
#pragma unroll
    for (int s = 0; s < NA; s++) st(j + NB * s, z[s]);
}

// radix of the register butterfly for an axis of length n (1: direct sum)
static inline int pw_pick_na(int n) { return n % 12 == 0 ? 12 : n % 8 == 0 ? 8 : 1; }

// x axis: T1[b][j1][c] = sum_q1i Cbox[q1i][c] exp(+2 pi i q1 j1 / N1); c = q2i nq3 + q3i a box column,
// table[q1i ncol + c] = index of that plane wave in C (or -1: outside the coefficient sphere).  One thread = one
// (column, j < N1/NA): nq1 twiddled terms and one radix-NA butterfly give its NA planes j + (N1/NA) s.
// grid (ceil(ncol/128), N1/NA, bands), block 128; consecutive threads = consecutive columns (coalesced table reads
// and T1 writes).
template <int NA>
__global__ void __launch_bounds__(128) pw_xaxis_kernel(const cd *__restrict__ C, int n_pw, const int32_t *__restrict__ table,
                                                      const cd *__restrict__ tw1, int N1, int q1min, int nq1, int ncol,
                                                      cd *__restrict__ T1) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncol) return;
    const int j = blockIdx.y, b = blockIdx.z;
    const cd *Cb = C + (size_t)b * n_pw;
    cd *Tb = T1 + (size_t)b * N1 * ncol + c;
    pw_expand_line<NA>(N1, j, q1min, nq1, tw1,
                       [&](int qi) {
                           const int idx = table[(size_t)qi * ncol + c];
                           return idx >= 0 ? Cb[idx] : cmake(0.0, 0.0);
                       },
                       [&](int n, cd v) { Tb[(size_t)n * ncol] = v; });
}

typedef void (*PwXKernel)(const cd *, int, const int32_t *, const cd *, int, int, int, int, cd *);
static inline PwXKernel pw_xaxis_pick(int na) { return na == 12 ? pw_xaxis_kernel<12> : na == 8 ? pw_xaxis_kernel<8> : pw_xaxis_kernel<1>; }

// One CTA per (x-plane j1, band).  Shared memory (cd): tw2[N2] | tw3[N3] | P[nq2][nq3] | Y[N2][nq3].
//   y: Y[.][q3i] from the box column P[.][q3i]   (task = (j < N2/NA2, q3i))
//   z: u[j2][.]  from the row Y[j2][.]           (task = (j2, j < N3/NA3); the NA3 stores of a task are 16 bytes at a
//      stride of N3/NA3 elements, consecutive j -> consecutive addresses)
template <int NA2, int NA3>
__global__ void __launch_bounds__(128, 3) pw_zy_kernel(const cd *__restrict__ T1, const cd *__restrict__ tw2,
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
    const int NB2 = N2 / NA2, NB3 = N3 / NA3;
    for (int i = tid; i < NB2 * nq3; i += nth) {
        const int j = i / nq3, c3 = i - j * nq3;
        pw_expand_line<NA2>(N2, j, q2min, nq2, tw2s, [&](int qi) { return P[qi * nq3 + c3]; },
                            [&](int n, cd v) { Y[n * nq3 + c3] = v; });
    }
    __syncthreads();
    cd *op = out + ((size_t)b * N1 + j1) * N2 * N3;
    for (int i = tid; i < N2 * NB3; i += nth) {
        const int j2 = i / NB3, j = i - j2 * NB3;
        const cd *yr = Y + (size_t)j2 * nq3;
        cd *orow = op + (size_t)j2 * N3;
        pw_expand_line<NA3>(N3, j, q3min, nq3, tw3s, [&](int qi) { return yr[qi]; }, [&](int n, cd v) { orow[n] = v; });
    }
}

// Table-driven variant for NA2, NA3 in {8, 12} (all BASELINE.json grids): persistent CTAs loop over (band, x-plane)
// items.  The twiddle of a term depends on (box position, j) only, so each CTA builds TWy[qi2][j < N2/NA2] and
// TWz[qi3][j < N3/NA3] once; the box is embedded in zero-padded arrays aligned to the radix (position = q - q0,
// q0 = qmin - (qmin mod NA)), so the inner loops have no bounds tests, no index updates and no conjugations: per term
// two LDS.128 with immediate offsets and one complex FMA.  The inverse butterfly is the forward one read at -s.
// Shared memory (cd): TWy[nq2p][NB2] | TWz[nq3p][NB3] | Pp[nq2p][nq3p] | Y[N2][nq3p + 1] (odd pitch in units of 16 bytes: the
// threads of a warp read the same element of four different rows in the z stage).
struct PwTabDims {
    int r2, nq2p, r3, nq3p;
    size_t smem;
};
static inline PwTabDims pw_tab_dims(int N2, int N3, int na2, int na3, int q2min, int nq2, int q3min, int nq3) {
    PwTabDims d;
    d.r2 = ((q2min % na2) + na2) % na2;
    d.r3 = ((q3min % na3) + na3) % na3;
    d.nq2p = (nq2 + d.r2 + na2 - 1) / na2 * na2;
    d.nq3p = (nq3 + d.r3 + na3 - 1) / na3 * na3;
    d.smem = ((size_t)d.nq2p * (N2 / na2) + (size_t)d.nq3p * (N3 / na3) + (size_t)d.nq2p * d.nq3p + (size_t)N2 * (d.nq3p + 1)) * sizeof(cd);
    return d;
}

template <int NA2, int NA3, int RY, int RZ>
__global__ void __launch_bounds__(128) pw_zy_tab_kernel(const cd *__restrict__ T1, const cd *__restrict__ tw2,
                                                       const cd *__restrict__ tw3, int N1, int N2, int N3, int q2min, int nq2,
                                                       int q3min, int nq3, int n_items, cd *__restrict__ out) {
    extern __shared__ __align__(16) unsigned char pw_smem[];
    const int NB2 = N2 / NA2, NB3 = N3 / NA3;
    const int r2 = ((q2min % NA2) + NA2) % NA2, r3 = ((q3min % NA3) + NA3) % NA3;
    const int nq2p = (nq2 + r2 + NA2 - 1) / NA2 * NA2, nq3p = (nq3 + r3 + NA3 - 1) / NA3 * NA3;
    cd *TWy = reinterpret_cast<cd *>(pw_smem);
    cd *TWz = TWy + nq2p * NB2;
    cd *Pp = TWz + nq3p * NB3;
    cd *Y = Pp + nq2p * nq3p;
    const int tid = threadIdx.x, nth = blockDim.x;
    for (int i = tid; i < nq2p * NB2; i += nth) {
        const int qi = i / NB2, j = i - qi * NB2;
        int t = (int)(((int64_t)(q2min - r2 + qi) * j) % N2);
        if (t < 0) t += N2;
        const cd w = tw2[t];                       // exp(-2 pi i t/N2): the inverse transform takes the conjugate
        TWy[i] = cmake(w.x, -w.y);
    }
    for (int i = tid; i < nq3p * NB3; i += nth) {
        const int qi = i / NB3, j = i - qi * NB3;
        int t = (int)(((int64_t)(q3min - r3 + qi) * j) % N3);
        if (t < 0) t += N3;
        const cd w = tw3[t];
        TWz[i] = cmake(w.x, -w.y);
    }
    const int yp = nq3p + 1;
    for (int i = tid; i < nq2p * nq3p + N2 * yp; i += nth) Pp[i] = cmake(0.0, 0.0);   // Pp and Y: the padding stays zero
    __syncthreads();
    const int ncol = nq2 * nq3;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const cd *Tp = T1 + (size_t)item * ncol;   // item = band * N1 + j1
        for (int i = tid; i < ncol; i += nth) {
            const int a = i / nq3, c = i - a * nq3;
            Pp[(r2 + a) * nq3p + r3 + c] = Tp[i];
        }
        __syncthreads();   // Pp complete; every thread has left the z stage of the previous item
        // y stage: RY values of j per thread (j, j + ceil(NB2 / RY), ...) share the loads of the box column; the z stage:
        // RZ rows j2 per thread share the twiddles.  One LDS.128 per operand and term was what bound the kernel (LSU pipe
        // 85 % busy, profiles/r2a): (1 + R) / R loads per complex multiply-add instead of 2.
        const int HB2 = (NB2 + RY - 1) / RY;
        for (int i = tid; i < HB2 * nq3; i += nth) {
            const int j0 = i / nq3, col = r3 + (i - j0 * nq3);
            cd z[RY][NA2];
            const cd *twp[RY];
#pragma unroll
            for (int r = 0; r < RY; r++) {
                twp[r] = TWy + min(j0 + r * HB2, NB2 - 1);   // a j beyond the axis repeats the last one and is not stored
#pragma unroll
                for (int k1 = 0; k1 < NA2; k1++) z[r][k1] = cmake(0.0, 0.0);
            }
            const cd *pp = Pp + col;
            for (int base = 0; base < nq2p; base += NA2) {
#pragma unroll
                for (int k1 = 0; k1 < NA2; k1++) {
                    const cd v = pp[(base + k1) * nq3p];
#pragma unroll
                    for (int r = 0; r < RY; r++) z[r][k1] = cfma(twp[r][(base + k1) * NB2], v, z[r][k1]);
                }
            }
#pragma unroll
            for (int r = 0; r < RY; r++) {
                const int j = j0 + r * HB2;
                if (j < NB2) {
                    Bfly<NA2>::run(z[r]);
#pragma unroll
                    for (int s = 0; s < NA2; s++) Y[(j + NB2 * ((NA2 - s) % NA2)) * yp + col] = z[r][s];
                }
            }
        }
        __syncthreads();
        cd *op = out + (size_t)item * N2 * N3;
        const int H2 = (N2 + RZ - 1) / RZ;
        for (int i = tid; i < H2 * NB3; i += nth) {
            const int j2 = i / NB3, j = i - j2 * NB3;
            cd z[RZ][NA3];
            const cd *yr[RZ];
#pragma unroll
            for (int r = 0; r < RZ; r++) {
                yr[r] = Y + (size_t)min(j2 + r * H2, N2 - 1) * yp;
#pragma unroll
                for (int k1 = 0; k1 < NA3; k1++) z[r][k1] = cmake(0.0, 0.0);
            }
            const cd *twp = TWz + j;
            for (int base = 0; base < nq3p; base += NA3) {
#pragma unroll
                for (int k1 = 0; k1 < NA3; k1++) {
                    const cd w = twp[(base + k1) * NB3];
#pragma unroll
                    for (int r = 0; r < RZ; r++) z[r][k1] = cfma(w, yr[r][base + k1], z[r][k1]);
                }
            }
#pragma unroll
            for (int r = 0; r < RZ; r++) {
                const int row = j2 + r * H2;
                if (row < N2) {
                    Bfly<NA3>::run(z[r]);
                    cd *orow = op + (size_t)row * N3 + j;
#pragma unroll
                    for (int s = 0; s < NA3; s++) orow[NB3 * ((NA3 - s) % NA3)] = z[r][s];
                }
            }
        }
    }
}

typedef void (*PwZyTabKernel)(const cd *, const cd *, const cd *, int, int, int, int, int, int, int, int, cd *);
static inline PwZyTabKernel pw_zy_tab_pick(int N2, int N3) {
    const int a2 = pw_pick_na(N2), a3 = pw_pick_na(N3);
    // register blocking (2 values of j in the y stage, 4 rows in the z stage) only where a plane still has tasks for
    // every thread afterwards: on the 24 x 24 planes of configs[2] (72 z tasks) it halves the speed, on 60 x 64 and
    // 40 x 168 it gains 8 - 15 %
    const bool blocked = a3 > 0 && N2 * (N3 / a3) >= 256;
#define PW_TAB_PICK(A2, A3) if (a2 == A2 && a3 == A3) return blocked ? pw_zy_tab_kernel<A2, A3, 2, 4> : pw_zy_tab_kernel<A2, A3, 1, 1>
    PW_TAB_PICK(12, 12);
    PW_TAB_PICK(12, 8);
    PW_TAB_PICK(8, 12);
    PW_TAB_PICK(8, 8);
#undef PW_TAB_PICK
    return nullptr;   // an axis without radix 8 or 12: pw_zy_kernel
}

typedef void (*PwZyKernel)(const cd *, const cd *, const cd *, int, int, int, int, int, int, int, cd *);
static inline PwZyKernel pw_zy_pick(int N2, int N3) {
    const int a2 = pw_pick_na(N2), a3 = pw_pick_na(N3);
    if (a2 == 12 && a3 == 12) return pw_zy_kernel<12, 12>;
    if (a2 == 12 && a3 == 8) return pw_zy_kernel<12, 8>;
    if (a2 == 8 && a3 == 12) return pw_zy_kernel<8, 12>;
    if (a2 == 8 && a3 == 8) return pw_zy_kernel<8, 8>;
    if (a2 == 12) return pw_zy_kernel<12, 1>;
    if (a2 == 8) return pw_zy_kernel<8, 1>;
    if (a3 == 12) return pw_zy_kernel<1, 12>;
    if (a3 == 8) return pw_zy_kernel<1, 8>;
    return pw_zy_kernel<1, 1>;
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
