/*
 * rpa_oracle.c -- CPU ORACLE for the chi0 / RPA hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, double-precision restatement of what the path computes, written from the paper
 * (P:Lnnn = /root/reference/PAPER.md line nnn) and the readings listed in DESIGN.md section 3.
 * It shares no code, header, table generator or helper with the CUDA library; only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Every function below is pinned by tests/test_oracle_pins.py (closed forms, library special
 * cases, brute force, invariants); none is "parity unpinned".
 *
 * Conventions: Hartree atomic units; cell rows a1,a2,a3; B = 2 pi A^-T;
 * K_g = (q_red + g) B; grid index j = (j1*N2 + j2)*N3 + j3 (C order); orbitals are the periodic
 * parts u(r_j), grid-normalised (1/N) sum |u|^2 = 1; complex128 interleaved.
 *
 * No blocking, no butterflies, no BLAS: direct sums only.  OpenMP only spreads independent
 * output elements over cores; it never changes the order of any single sum.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double _Complex zd;

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* B = 2 pi A^-T  (a_i . b_j = 2 pi delta_ij), plain cofactor inverse. */
static void recip_cell(const double A[9], double B[9]) {
    const double a = A[0], b = A[1], c = A[2], d = A[3], e = A[4], f = A[5], g = A[6], h = A[7], i = A[8];
    const double det = a * (e * i - f * h) - b * (d * i - f * g) + c * (d * h - e * g);
    const double s = 2.0 * M_PI / det;
    /* inverse(A)[r][c] = cof[c][r]/det ; B = 2pi * inverse(A)^T  => B[r][c] = 2pi*cof[r][c]/det */
    B[0] = s * (e * i - f * h);
    B[1] = s * -(d * i - f * g);
    B[2] = s * (d * h - e * g);
    B[3] = s * -(b * i - c * h);
    B[4] = s * (a * i - c * g);
    B[5] = s * -(a * h - b * g);
    B[6] = s * (b * f - c * e);
    B[7] = s * -(a * f - c * d);
    B[8] = s * (a * e - b * d);
}

double orc_volume(const double A[9]) {
    const double det = A[0] * (A[4] * A[8] - A[5] * A[7]) - A[1] * (A[3] * A[8] - A[5] * A[6]) +
                       A[2] * (A[3] * A[7] - A[4] * A[6]);
    return fabs(det);
}

/* K_g = (q_red + g) B, Cartesian (bohr^-1). */
static void kvec(const double B[9], const double q[3], const int32_t g[3], double K[3]) {
    const double x = q[0] + g[0], y = q[1] + g[1], z = q[2] + g[2];
    K[0] = x * B[0] + y * B[3] + z * B[6];
    K[1] = x * B[1] + y * B[4] + z * B[7];
    K[2] = x * B[2] + y * B[5] + z * B[8];
}

/*
 * Step 1, the G sphere ("size ... defined by a cutoff energy", Table 1 step 6; readings A6, A7):
 * all integer g with |g_i| < N_i/2 (strict) and |K_g|^2/2 <= ecut, ordered by ascending flat FFT index
 * ((g1 mod N1)*N2 + (g2 mod N2))*N3 + (g3 mod N3).  Returns ng (also when ng > max_ng; then nothing beyond
 * max_ng is written).  g_out[ng][3], K2_out[ng] = |K_g|^2 (either may be NULL).
 */
int32_t orc_sphere(const int32_t grid[3], const double cell[9], const double q_red[3], double ecut_ha,
                   int32_t max_ng, int32_t *g_out, double *K2_out) {
    double B[9];
    recip_cell(cell, B);
    int32_t ng = 0;
    for (int32_t i1 = 0; i1 < grid[0]; i1++)
        for (int32_t i2 = 0; i2 < grid[1]; i2++)
            for (int32_t i3 = 0; i3 < grid[2]; i3++) {
                /* walking i1,i2,i3 in C order IS ascending flat FFT index */
                int32_t g[3];
                g[0] = (2 * i1 < grid[0]) ? i1 : i1 - grid[0];
                g[1] = (2 * i2 < grid[1]) ? i2 : i2 - grid[1];
                g[2] = (2 * i3 < grid[2]) ? i3 : i3 - grid[2];
                if (2 * abs(g[0]) >= grid[0] || 2 * abs(g[1]) >= grid[1] || 2 * abs(g[2]) >= grid[2]) continue;
                double K[3];
                kvec(B, q_red, g, K);
                const double K2 = K[0] * K[0] + K[1] * K[1] + K[2] * K[2];
                if (0.5 * K2 <= ecut_ha) {
                    if (ng < max_ng) {
                        if (g_out) { g_out[3 * ng] = g[0]; g_out[3 * ng + 1] = g[1]; g_out[3 * ng + 2] = g[2]; }
                        if (K2_out) K2_out[ng] = K2;
                    }
                    ng++;
                }
            }
    return ng;
}

/* |K_g|^2 for an arbitrary list of g (used for sampled sub-lists). */
void orc_K2(const double cell[9], const double q_red[3], int32_t ng, const int32_t *g, double *K2_out) {
    double B[9];
    recip_cell(cell, B);
    for (int32_t i = 0; i < ng; i++) {
        double K[3];
        kvec(B, q_red, g + 3 * i, K);
        K2_out[i] = K[0] * K[0] + K[1] * K[1] + K[2] * K[2];
    }
}

/* exp(-2 pi i t / n), t = 0..n-1, evaluated in long double (reading: step 2 of SURVEY 8(c)). */
static zd *phase_table(int32_t n) {
    zd *t = (zd *)malloc(sizeof(zd) * (size_t)n);
    for (int32_t k = 0; k < n; k++) {
        const long double a = -2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)n;
        t[k] = (double)cosl(a) + (double)sinl(a) * I;
    }
    return t;
}

static inline int32_t pmod(int64_t a, int32_t n) {
    int64_t r = a % n;
    return (int32_t)(r < 0 ? r + n : r);
}

/*
 * Step 2, naive mode: the literal triple sum of Eq. 7 / Eq. 12 (readings A4, A5):
 *   ntilde_nm(g) = (1/N) sum_{j1 j2 j3} conj(u_n[j]) u_m[j] exp(-2 pi i (g1 j1/N1 + g2 j2/N2 + g3 j3/N3))
 * for each g of the list, for each of n_m orbitals u_m against ONE u_n.  out[m][g].
 */
void orc_pair_density_naive(const int32_t grid[3], const zd *u_n, int32_t n_m, const zd *u_m, int32_t ng,
                            const int32_t *g, zd *out) {
    const int32_t N1 = grid[0], N2 = grid[1], N3 = grid[2];
    const int64_t N = (int64_t)N1 * N2 * N3;
    zd *t1 = phase_table(N1), *t2 = phase_table(N2), *t3 = phase_table(N3);
#pragma omp parallel for collapse(2) schedule(dynamic)
    for (int32_t m = 0; m < n_m; m++)
        for (int32_t ig = 0; ig < ng; ig++) {
            const int32_t g1 = g[3 * ig], g2 = g[3 * ig + 1], g3 = g[3 * ig + 2];
            const zd *um = u_m + (int64_t)m * N;
            zd acc = 0.0;
            for (int32_t j1 = 0; j1 < N1; j1++)
                for (int32_t j2 = 0; j2 < N2; j2++)
                    for (int32_t j3 = 0; j3 < N3; j3++) {
                        const int64_t j = ((int64_t)j1 * N2 + j2) * N3 + j3;
                        const zd ph = t1[pmod((int64_t)g1 * j1, N1)] * t2[pmod((int64_t)g2 * j2, N2)] *
                                      t3[pmod((int64_t)g3 * j3, N3)];
                        acc += conj(u_n[j]) * um[j] * ph;
                    }
            out[(int64_t)m * ng + ig] = acc / (double)N;
        }
    free(t1); free(t2); free(t3);
}

/*
 * Step 2, separable mode: the same sum, evaluated as three nested 1-D direct sums restricted to the g3, g2, g1
 * values present in the list (the exponential factorises; still no butterflies).  out[m][g].
 */
void orc_pair_density_separable(const int32_t grid[3], const zd *u_n, int32_t n_m, const zd *u_m, int32_t ng,
                                const int32_t *g, zd *out) {
    const int32_t N1 = grid[0], N2 = grid[1], N3 = grid[2];
    const int64_t N = (int64_t)N1 * N2 * N3;
    zd *t1 = phase_table(N1), *t2 = phase_table(N2), *t3 = phase_table(N3);
    /* distinct g2, g3 values in the list, as compact index maps */
    int32_t *map2 = (int32_t *)malloc(sizeof(int32_t) * (size_t)N2), *map3 = (int32_t *)malloc(sizeof(int32_t) * (size_t)N3);
    int32_t *val2 = (int32_t *)malloc(sizeof(int32_t) * (size_t)N2), *val3 = (int32_t *)malloc(sizeof(int32_t) * (size_t)N3);
    int32_t n2 = 0, n3 = 0;
    for (int32_t i = 0; i < N2; i++) map2[i] = -1;
    for (int32_t i = 0; i < N3; i++) map3[i] = -1;
    for (int32_t ig = 0; ig < ng; ig++) {
        const int32_t r2 = pmod(g[3 * ig + 1], N2), r3 = pmod(g[3 * ig + 2], N3);
        if (map2[r2] < 0) { map2[r2] = n2; val2[n2++] = g[3 * ig + 1]; }
        if (map3[r3] < 0) { map3[r3] = n3; val3[n3++] = g[3 * ig + 2]; }
    }
#pragma omp parallel
    {
        zd *Abuf = (zd *)malloc(sizeof(zd) * (size_t)N1 * N2 * n3);
        zd *Bbuf = (zd *)malloc(sizeof(zd) * (size_t)N1 * n2 * n3);
#pragma omp for schedule(dynamic)
        for (int32_t m = 0; m < n_m; m++) {
            const zd *um = u_m + (int64_t)m * N;
            /* a: A[j1][j2][c3] = sum_j3 conj(u_n) u_m exp(-2 pi i g3 j3 / N3) */
            for (int32_t j1 = 0; j1 < N1; j1++)
                for (int32_t j2 = 0; j2 < N2; j2++) {
                    const int64_t base = ((int64_t)j1 * N2 + j2) * N3;
                    for (int32_t c3 = 0; c3 < n3; c3++) {
                        zd acc = 0.0;
                        for (int32_t j3 = 0; j3 < N3; j3++)
                            acc += conj(u_n[base + j3]) * um[base + j3] * t3[pmod((int64_t)val3[c3] * j3, N3)];
                        Abuf[((int64_t)j1 * N2 + j2) * n3 + c3] = acc;
                    }
                }
            /* b: B[j1][c2][c3] = sum_j2 A[j1][j2][c3] exp(-2 pi i g2 j2 / N2) */
            for (int32_t j1 = 0; j1 < N1; j1++)
                for (int32_t c2 = 0; c2 < n2; c2++)
                    for (int32_t c3 = 0; c3 < n3; c3++) {
                        zd acc = 0.0;
                        for (int32_t j2 = 0; j2 < N2; j2++)
                            acc += Abuf[((int64_t)j1 * N2 + j2) * n3 + c3] * t2[pmod((int64_t)val2[c2] * j2, N2)];
                        Bbuf[((int64_t)j1 * n2 + c2) * n3 + c3] = acc;
                    }
            /* c: out[g] = (1/N) sum_j1 B[j1][c2(g)][c3(g)] exp(-2 pi i g1 j1 / N1) */
            for (int32_t ig = 0; ig < ng; ig++) {
                const int32_t g1 = g[3 * ig];
                const int32_t c2 = map2[pmod(g[3 * ig + 1], N2)], c3 = map3[pmod(g[3 * ig + 2], N3)];
                zd acc = 0.0;
                for (int32_t j1 = 0; j1 < N1; j1++)
                    acc += Bbuf[((int64_t)j1 * n2 + c2) * n3 + c3] * t1[pmod((int64_t)g1 * j1, N1)];
                out[(int64_t)m * ng + ig] = acc / (double)N;
            }
        }
        free(Abuf); free(Bbuf);
    }
    free(map2); free(map3); free(val2); free(val3);
    free(t1); free(t2); free(t3);
}

/*
 * Step 3, PAW one-centre correction (Eq. 6; Table 1 steps 8-9; readings A8, A9, A10):
 *   n_nm(g) += sum_a exp(-i K_g . R_a) sum_{i,j} conj(P^a_{i,n}) Q^a_{ij}(g) P^a_{j,m}
 * P_n[sum n_proj] for the ONE occupied band, P_m[n_m][sum n_proj]; Q per atom [n_i][n_i][ng], atoms
 * concatenated; R_cart[n_atoms][3].  n[m][g] updated in place.  Q is a general complex matrix in (i,j).
 */
void orc_paw_add(const double cell[9], const double q_red[3], int32_t ng, const int32_t *g, int32_t n_atoms,
                 const int32_t *n_proj, const zd *P_n, int32_t n_m, const zd *P_m, const zd *Q, const double *R_cart,
                 zd *n) {
    double B[9];
    recip_cell(cell, B);
    int32_t ptot = 0;
    for (int32_t a = 0; a < n_atoms; a++) ptot += n_proj[a];
#pragma omp parallel for collapse(2) schedule(static)
    for (int32_t m = 0; m < n_m; m++)
        for (int32_t ig = 0; ig < ng; ig++) {
            double K[3];
            kvec(B, q_red, g + 3 * ig, K);
            zd corr = 0.0;
            int64_t qoff = 0;
            int32_t poff = 0;
            for (int32_t a = 0; a < n_atoms; a++) {
                const int32_t ni = n_proj[a];
                const double kr = K[0] * R_cart[3 * a] + K[1] * R_cart[3 * a + 1] + K[2] * R_cart[3 * a + 2];
                const zd ph = cos(kr) - sin(kr) * I;
                zd s = 0.0;
                for (int32_t i = 0; i < ni; i++)
                    for (int32_t j = 0; j < ni; j++)
                        s += conj(P_n[poff + i]) * Q[qoff + ((int64_t)i * ni + j) * ng + ig] *
                             P_m[(int64_t)m * ptot + poff + j];
                corr += ph * s;
                qoff += (int64_t)ni * ni * ng;
                poff += ni;
            }
            n[(int64_t)m * ng + ig] += corr;
        }
}

/*
 * Step 4, transition weights (Eq. 18 in the real form of BASELINE.json north_star; readings A1, A12):
 *   w_nm(omega) = 2 (f_n - f_m)(eps_n - eps_m) / (omega^2 + (eps_n - eps_m)^2),   one occupied n, n_m unoccupied.
 * w[iw][m].
 */
void orc_weights(double eps_n, double f_n, int32_t n_m, const double *eps_m, const double *f_m, int32_t n_omega,
                 const double *omega, double *w) {
    for (int32_t iw = 0; iw < n_omega; iw++)
        for (int32_t m = 0; m < n_m; m++) {
            const double de = eps_n - eps_m[m];
            w[(int64_t)iw * n_m + m] = 2.0 * (f_n - f_m[m]) * de / (omega[iw] * omega[iw] + de * de);
        }
}

/*
 * Step 5, accumulation by explicit rank-1 sums (Eq. 17): for every omega and EVERY (g,g') -- both
 * triangles, independently --
 *   S_w[g][g'] += kweight * sum_p w[iw][p] n_p(g) conj(n_p(g')),   p ascending.
 * n[p][g] (n_p pairs), w[iw][p], S[n_omega][ng][ng].
 */
void orc_accumulate(int32_t ng, int32_t n_p, const zd *n, int32_t n_omega, const double *w, double kweight, zd *S) {
#pragma omp parallel for collapse(2) schedule(static)
    for (int32_t iw = 0; iw < n_omega; iw++)
        for (int32_t a = 0; a < ng; a++) {
            zd *row = S + ((int64_t)iw * ng + a) * ng;
            for (int32_t b = 0; b < ng; b++) {
                zd acc = 0.0;
                for (int32_t p = 0; p < n_p; p++)
                    acc += w[(int64_t)iw * n_p + p] * n[(int64_t)p * ng + a] * conj(n[(int64_t)p * ng + b]);
                row[b] += kweight * acc;
            }
        }
}

/*
 * SURVEY 8(f) NEXT-4, second workload ("the non-interacting response function is one key ingredient" of
 * TDDFT / GW / BSE): Eq. 3 at a general complex frequency z in place of i omega (z = omega + i eta on the
 * real axis), reading A19.  Eq. 3 sums over BOTH orderings of every band pair; under time reversal the
 * reversed ordering (m -> n) has the same n n^H as (n -> m) (reading A1), so for one occupied n and n_m unoccupied m
 *   w_nm(z) = (f_n - f_m) / (z + eps_n - eps_m)  +  (f_m - f_n) / (z + eps_m - eps_n)        (complex),
 * each term written as printed.  w[iz][m].
 */
void orc_weights_z(double eps_n, double f_n, int32_t n_m, const double *eps_m, const double *f_m, int32_t n_z,
                   const zd *z, zd *w) {
    for (int32_t iz = 0; iz < n_z; iz++)
        for (int32_t m = 0; m < n_m; m++) {
            const zd forward = (f_n - f_m[m]) / (z[iz] + eps_n - eps_m[m]);
            const zd reversed = (f_m[m] - f_n) / (z[iz] + eps_m[m] - eps_n);
            w[(int64_t)iz * n_m + m] = forward + reversed;
        }
}

/* Eq. 17 with those complex weights: S_z[g][g'] += kweight * sum_p w[iz][p] n_p(g) conj(n_p(g')). */
void orc_accumulate_z(int32_t ng, int32_t n_p, const zd *n, int32_t n_z, const zd *w, double kweight, zd *S) {
#pragma omp parallel for collapse(2) schedule(static)
    for (int32_t iz = 0; iz < n_z; iz++)
        for (int32_t a = 0; a < ng; a++) {
            zd *row = S + ((int64_t)iz * ng + a) * ng;
            for (int32_t b = 0; b < ng; b++) {
                zd acc = 0.0;
                for (int32_t p = 0; p < n_p; p++)
                    acc += w[(int64_t)iz * n_p + p] * (n[(int64_t)p * ng + a] * conj(n[(int64_t)p * ng + b]));
                row[b] += kweight * acc;
            }
        }
}

/* Step 6, prefactor of Eq. 3 (readings A1-A3): chi0 = (2/Omega) S, spin-paired. */
void orc_chi0_from_S(int64_t count, double volume, const zd *S, zd *chi0) {
    const double s = 2.0 / volume;
    for (int64_t i = 0; i < count; i++) chi0[i] = s * S[i];
}

/*
 * Step 7, per-q energy (Eq. 1-2, Table 1 step 13 P:L161; readings A14, A17):
 *   X = D chi0 D, D = diag(sqrt(v));  e(w) = ln det(I - X) + Tr X via textbook unblocked Cholesky of the
 *   Hermitian positive-definite I - X: ln det = 2 sum ln L_ii;   E_c(q) = (1/2pi) sum_i wt_i e(w_i).
 * chi0[n_omega][ng][ng]; e_omega[n_omega] optional.  Returns 0, or -(iw+1) if I - X is not positive definite.
 */
int32_t orc_ec_q(int32_t ng, int32_t n_omega, const zd *chi0, const double *v, const double *omega_wt, double *ec_out,
                 double *e_omega) {
    int32_t status = 0;
    double *e = (double *)malloc(sizeof(double) * (size_t)n_omega);
#pragma omp parallel for schedule(dynamic)
    for (int32_t iw = 0; iw < n_omega; iw++) {
        zd *M = (zd *)malloc(sizeof(zd) * (size_t)ng * ng);
        const zd *c = chi0 + (int64_t)iw * ng * ng;
        double trX = 0.0;
        for (int32_t a = 0; a < ng; a++)
            for (int32_t b = 0; b < ng; b++) {
                const zd x = sqrt(v[a]) * c[(int64_t)a * ng + b] * sqrt(v[b]);
                if (a == b) trX += creal(x);
                M[(int64_t)a * ng + b] = (a == b ? 1.0 : 0.0) - x;
            }
        /* Cholesky-Banachiewicz, lower triangle, row by row */
        double logdet = 0.0;
        int bad = 0;
        for (int32_t a = 0; a < ng && !bad; a++) {
            for (int32_t b = 0; b <= a; b++) {
                zd s = M[(int64_t)a * ng + b];
                for (int32_t k = 0; k < b; k++) s -= M[(int64_t)a * ng + k] * conj(M[(int64_t)b * ng + k]);
                if (a == b) {
                    const double d = creal(s);
                    if (!(d > 0.0)) { bad = 1; break; }
                    M[(int64_t)a * ng + a] = sqrt(d);
                    logdet += 2.0 * log(sqrt(d));
                } else {
                    M[(int64_t)a * ng + b] = s / creal(M[(int64_t)b * ng + b]);
                }
            }
        }
        if (bad) {
#pragma omp critical
            status = -(iw + 1);
            e[iw] = NAN;
        } else {
            e[iw] = logdet + trX;
        }
        free(M);
    }
    double ec = 0.0;
    for (int32_t iw = 0; iw < n_omega; iw++) {
        ec += omega_wt[iw] * e[iw];
        if (e_omega) e_omega[iw] = e[iw];
    }
    *ec_out = ec / (2.0 * M_PI);
    free(e);
    return status;
}

/*
 * ---- NEXT-1: Table 1 steps 3-4 -----------------------------------------------------------------
 * Eq. 10: the periodic part of the pseudo wave function on the grid from its plane-wave coefficients,
 *   u(r_j) = sum_Q C(Q) exp(+2 pi i (Q1 j1/N1 + Q2 j2/N2 + Q3 j3/N3)),
 * by direct summation (the Bloch phase exp(i k.r) of Eq. 10 is not applied: reading A5, the library works with
 * periodic parts).  Evaluated at the n_pts grid points listed in pts (flat C-order indices); out[band][pt].
 * No normalisation: (1/N) sum_j |u_j|^2 = sum_Q |C(Q)|^2 (Parseval) is the caller's.
 */
void orc_pw_to_grid(const int32_t grid[3], int32_t n_bands, int32_t n_pw, const int32_t *g_pw, const zd *C,
                    int64_t n_pts, const int64_t *pts, zd *out) {
    const int32_t N1 = grid[0], N2 = grid[1], N3 = grid[2];
    zd *t1 = phase_table(N1), *t2 = phase_table(N2), *t3 = phase_table(N3);
#pragma omp parallel for collapse(2) schedule(dynamic, 64)
    for (int32_t b = 0; b < n_bands; b++)
        for (int64_t ip = 0; ip < n_pts; ip++) {
            const int64_t j = pts[ip];
            const int32_t j3 = (int32_t)(j % N3), j2 = (int32_t)((j / N3) % N2), j1 = (int32_t)(j / ((int64_t)N2 * N3));
            zd acc = 0.0;
            for (int32_t q = 0; q < n_pw; q++) {
                /* exp(+2 pi i t/n) = conj(exp(-2 pi i t/n)) */
                const zd ph = conj(t1[pmod((int64_t)g_pw[3 * q] * j1, N1)] * t2[pmod((int64_t)g_pw[3 * q + 1] * j2, N2)] *
                                   t3[pmod((int64_t)g_pw[3 * q + 2] * j3, N3)]);
                acc += C[(int64_t)b * n_pw + q] * ph;
            }
            out[(int64_t)b * n_pts + ip] = acc;
        }
    free(t1); free(t2); free(t3);
}

/*
 * Eq. 11: IBZ -> BZ transformation of the periodic part on the grid,
 *   u_out(r) = u_in(T^-1 r)            (crystal symmetry),     then conj if time reversal is used,
 * with T^-1 given in reduced (fractional) coordinates as the integer matrix M: a point with fractional
 * coordinates x_i = j_i/N_i is taken from x'_i = sum_k M[i][k] x_k, i.e. grid index j'_i = sum_k M[i][k] j_k N_i/N_k
 * (mod N_i), which must be an integer for every grid point (returns -1 otherwise, 0 on success).
 */
int32_t orc_symmetry_remap(const int32_t grid[3], const int32_t M[9], int32_t time_reversal, int32_t n_bands,
                           const zd *in, zd *out) {
    const int64_t N = (int64_t)grid[0] * grid[1] * grid[2];
    for (int i = 0; i < 3; i++)
        for (int k = 0; k < 3; k++)
            if (((int64_t)M[3 * i + k] * grid[i]) % grid[k] != 0) return -1;
    for (int32_t b = 0; b < n_bands; b++)
        for (int32_t j1 = 0; j1 < grid[0]; j1++)
            for (int32_t j2 = 0; j2 < grid[1]; j2++)
                for (int32_t j3 = 0; j3 < grid[2]; j3++) {
                    const int64_t j[3] = {j1, j2, j3};
                    int64_t jp[3];
                    for (int i = 0; i < 3; i++) {
                        int64_t s = 0;
                        for (int k = 0; k < 3; k++) s += (int64_t)M[3 * i + k] * grid[i] / grid[k] * j[k];
                        jp[i] = pmod(s, grid[i]);
                    }
                    const zd v = in[b * N + (jp[0] * grid[1] + jp[1]) * grid[2] + jp[2]];
                    out[b * N + ((int64_t)j1 * grid[1] + j2) * grid[2] + j3] = time_reversal ? conj(v) : v;
                }
    return 0;
}

/*
 * ---- NEXT-2: Table 1 step 10, the optical limit q -> 0 of the G = 0 element --------------------------
 * Eq. 15 with Eq. 19: matrix elements of the gradient between pseudo wave functions expanded
 * in plane waves on a common set {Q} (same k for n and m), plus the PAW term,
 *   grad[al][n][m] = sum_Q conj(C_n(Q)) i (k + Q B)_al C_m(Q)
 *                    + sum_a sum_ij conj(P^a_{i,n}) Qgrad^a_al[i][j] P^a_{j,m},          al = x, y, z,
 * with sum_Q |C(Q)|^2 = 1 <=> the wave functions normalised in the cell.  Qgrad (Eq. 16; printed as Q_ii, read as
 * Q_ij like reading A8) is an input: per atom [3][n_i][n_i], atoms concatenated.  Plain loops.
 */
void orc_momentum_pw(const double cell[9], const double k_cart[3], int32_t n_pw, const int32_t *g_pw, int32_t n_occ,
                     const zd *C_occ, int32_t n_unocc, const zd *C_unocc, int32_t n_atoms, const int32_t *n_proj,
                     const zd *P_occ, const zd *P_unocc, const zd *Qgrad, zd *grad) {
    double B[9];
    recip_cell(cell, B);
    int32_t ptot = 0;
    for (int32_t a = 0; a < n_atoms; a++) ptot += n_proj[a];
    for (int al = 0; al < 3; al++)
        for (int32_t n = 0; n < n_occ; n++)
            for (int32_t m = 0; m < n_unocc; m++) {
                zd acc = 0.0;
                for (int32_t q = 0; q < n_pw; q++) {
                    const double G = g_pw[3 * q] * B[al] + g_pw[3 * q + 1] * B[3 + al] + g_pw[3 * q + 2] * B[6 + al];
                    acc += conj(C_occ[(int64_t)n * n_pw + q]) * (I * (k_cart[al] + G)) * C_unocc[(int64_t)m * n_pw + q];
                }
                int32_t poff = 0;
                int64_t qoff = 0;
                for (int32_t a = 0; a < n_atoms; a++) {
                    const int32_t ni = n_proj[a];
                    for (int32_t i = 0; i < ni; i++)
                        for (int32_t j = 0; j < ni; j++)
                            acc += conj(P_occ[(int64_t)n * ptot + poff + i]) * Qgrad[qoff + ((int64_t)al * ni + i) * ni + j] *
                                   P_unocc[(int64_t)m * ptot + poff + j];
                    poff += ni;
                    qoff += (int64_t)3 * ni * ni;
                }
                grad[((int64_t)al * n_occ + n) * n_unocc + m] = acc;
            }
}

/*
 * Eq. 13 (printed twice, the second line is the result): the G = 0 pair density in the limit q -> 0 along
 * the unit vector qdir, per unit |q|,
 *   n_nm(G = 0) = -i qdir . grad[.][n][m] / (eps_m - eps_n),        0 when eps_m = eps_n (its weight is 0 anyway).
 * head[n][m].
 */
void orc_optical_head(int32_t n_occ, int32_t n_unocc, const double *eps_occ, const double *eps_unocc, const double qdir[3],
                      const zd *grad, zd *head) {
    for (int32_t n = 0; n < n_occ; n++)
        for (int32_t m = 0; m < n_unocc; m++) {
            const double de = eps_unocc[m] - eps_occ[n];
            zd s = 0.0;
            for (int al = 0; al < 3; al++) s += qdir[al] * grad[((int64_t)al * n_occ + n) * n_unocc + m];
            head[(int64_t)n * n_unocc + m] = de != 0.0 ? -I * s / de : 0.0;
        }
}

/*
 * NEXT-4: spin-polarised systems.  "The spin index sigma is implicitly contained" in Eq. 3 (
 * reading A3 fixed s = 2 for spin-paired bands): with explicit spin channels every channel is summed with degeneracy
 * s = 1, chi0 = (s/Omega) S.  Same as orc_chi0_from_S with the prefactor's 2 replaced by s.
 */
void orc_chi0_from_S_spin(int64_t count, double volume, double spin_deg, const zd *S, zd *chi0) {
    const double s = spin_deg / volume;
    for (int64_t i = 0; i < count; i++) chi0[i] = s * S[i];
}
