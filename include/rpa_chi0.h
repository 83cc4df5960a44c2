/*
 * rpa_chi0.h -- C ABI of the B200-native chi0 / RPA hot path (librpa_chi0.so).
 *
 * What it computes: the non-interacting density response chi0_GG'(q, i omega) of the RPA correlation energy
 * in the PAW method, and the per-q energy integrand, as stated in the paper
 * (P:Lnnn = /root/reference/PAPER.md line nnn):
 *
 *   pair density   ntilde_nm(G) = F[ conj(u_nk(r)) u_m,k+q(r) ]            Eq. 7 / Eq. 12
 *   PAW correction n_nm(G) = ntilde_nm(G) + sum_a e^{-i(q+G).R_a} sum_ij conj(P^a_i,n) Q^a_ij(q+G) P^a_j,m
 *                                                                           Eq. 6
 *   accumulation   chi0(i w) = (2/Omega) sum_k wk sum_{n occ, m unocc} w_nm(w) n_nm(G) conj(n_nm(G'))
 *                  w_nm(w) = 2 (f_n - f_m)(e_n - e_m) / (w^2 + (e_n - e_m)^2)   Eq. 3, 17, 18
 *   energy         E_c(q) = (1/2pi) sum_i wt_i { ln det[1 - v chi0(i w_i)] + Tr[v chi0(i w_i)] }
 *                                                                           Eq. 1-2
 *
 * Conventions: Hartree atomic units (bohr, Ha).  Grid N1 x N2 x N3, C order (index 3
 * fastest).  cell = rows a1,a2,a3; B = 2 pi cell^-T; K_g = (q_red + g) B for integer g.  Orbitals are the
 * cell-periodic parts u(r_j) on the grid, normalised (1/N) sum_j |u_j|^2 = 1.  complex128 is interleaved
 * (re, im) doubles ("cdouble").  Every G-indexed array (Q, v_G, chi0 rows/cols) is ordered as
 * rpa_chi0_gvectors() returns: ascending flat FFT index ((g1 mod N1) N2 + (g2 mod N2)) N3 + (g3 mod N3).
 *
 * Memory: "dev" pointers are CUDA device pointers (allocated by the caller, e.g. with PyTorch); "host"
 * pointers are ordinary host memory.  The library allocates no device memory: everything it needs is carved
 * from the caller's `workspace`.  All inputs are read-only and stay owned by the caller.
 *
 * Stream semantics: every call on a handle enqueues its work on the cudaStream_t given to rpa_chi0_create and
 * may return before the device work finishes; device inputs must stay alive until the stream reaches that
 * point.  Host input arrays are consumed before the call returns.  rpa_ec_q and rpa_chi0_sync block.
 *
 * Internal resources: besides the workspace the handle owns seven CUDA streams (used by rpa_ec_q: a high-priority
 * stream per lane for the look-ahead update, panels and strips, which run ahead of the big trailing updates, and a
 * main stream for each lane but the first, which uses the caller's; a lane factorises its share of the frequencies
 * concurrently with the others; all ordered with the caller's stream by events), a few events, two tensor maps over its
 * own workspace, and the CUDA graphs rpa_ec_q captures on first use (one per number of matrices in a group and lanes: the
 * factorisation is a few hundred small dependent launches, replayed with one launch), all released by rpa_chi0_destroy.
 *
 * Arithmetic: everything is FP64 / complex128 ("Double and double complex precision").  The rank-K accumulation
 * (Eq. 17 / Eq. 20) runs on the FP64 tensor cores (DMMA) by default; when that kernel splits K over several CTAs per
 * tile (chosen by the library) the tile sums use floating-point atomics: chi0 is then reproducible to rounding (~1e-16
 * relative), not bitwise.  rpa_chi0_set_rank_k_mode selects other kernels per handle, among them an opt-in int8-sliced
 * emulation with a stated error bound.  The library reads no environment variables and keeps no global state besides the
 * thread-local error string.
 *
 * Errors: every int-returning call gives 0 on success or a negative RPA_ERR_* code; rpa_last_error() holds
 * a thread-local message.  Nothing is thrown across the ABI.  A handle is not thread-safe; distinct handles
 * are independent.
 */
#ifndef RPA_CHI0_H
#define RPA_CHI0_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RPA_OK 0
#define RPA_ERR_INVALID_ARG (-1)  /* null pointer, non-positive size, omega <= 0, i_omega out of range, |K_g| = 0 */
#define RPA_ERR_UNSUPPORTED (-2)  /* unsupported grid length; plain add_kpoint on a q = 0 handle; grid-incompatible symmetry */
#define RPA_ERR_WORKSPACE (-3)    /* workspace too small or misaligned */
#define RPA_ERR_CUDA (-4)         /* a CUDA runtime call or kernel launch failed */
#define RPA_ERR_NOT_PD (-5)       /* 1 - v^1/2 chi0 v^1/2 not positive definite in rpa_ec_q */

typedef struct rpa_chi0 rpa_chi0_t; /* opaque, owned by the library, freed by rpa_chi0_destroy */

/*
 * Bytes of device workspace rpa_chi0_create needs for this sphere (Table 1 step 6) and omega count.
 * max_batch_pairs bounds how many (n,m) transitions are grouped into one batched pass (the paper's "Nu",
 * Eq. 20); <= 0 picks the default (8192).  Results never depend on it beyond rounding order.
 * max_proj_total bounds sum_a n_proj[a] of later rpa_chi0_add_kpoint calls (0: no PAW term will be used); it
 * sizes the scratch of the PAW contraction (Table 1 steps 8-9).
 * All pointers host.  Returns 0 on invalid arguments.
 */
size_t rpa_chi0_workspace_bytes(const int32_t grid[3], const double cell[9], const double q_red[3],
                                double ecut_ha, int32_t n_omega, int32_t max_batch_pairs, int32_t max_proj_total);

/*
 * Create a handle for one q: builds the |q+G|^2/2 <= ecut_ha sphere (strict |g_i| < N_i/2), its index
 * tables and the FFT twiddles, and zeroes the n_omega accumulators.
 *   grid, cell, q_red, omega_ha[n_omega] (> 0), omega_wt[n_omega] (may be NULL if rpa_ec_q is not used): host.
 *   workspace: dev, 256-byte aligned, at least rpa_chi0_workspace_bytes(...) bytes, must outlive the handle.
 *   cuda_stream: a cudaStream_t (NULL = legacy default stream).
 * q_red = 0 creates an optical-limit handle (pair densities then come from rpa_chi0_add_kpoint_optical).  A grid
 * length N2 or N3 with a prime factor other than 2, 3, 5, 7 (N1 is unrestricted), or a grid so large that one z line
 * per chunk does not fit shared memory, gives RPA_ERR_UNSUPPORTED.
 */
int rpa_chi0_create(rpa_chi0_t **out, const int32_t grid[3], const double cell[9], const double q_red[3],
                    double ecut_ha, int32_t n_omega, const double *omega_ha, const double *omega_wt,
                    int32_t max_batch_pairs, int32_t max_proj_total, void *workspace, size_t workspace_bytes,
                    void *cuda_stream);

/*
 * SURVEY 8(f) NEXT-4, second workload (chi0 as the ingredient of TDDFT / GW / BSE): the same chi0 on the REAL
 * frequency axis.  Eq. 3 is evaluated at z = omega + i eta instead of i omega, both orderings of each band
 * pair as printed, the reversed one folded onto the occ -> unocc pair by time reversal (readings A1, A19):
 *   chi0_GG'(omega) = (s/Omega) sum_k wk sum_{n occ, m unocc} w_nm(z) n_nm(G) conj(n_nm(G')),
 *   w_nm(z) = (f_n - f_m) [ 1/(z + e_n - e_m) - 1/(z + e_m - e_n) ]                 (complex; chi0 is not Hermitian).
 * The weight splits into real and imaginary parts, so the handle keeps TWO Hermitian accumulators per frequency and
 * every add_kpoint call runs the same kernels as on the imaginary axis over 2 n_omega slots:
 *   workspace: at least rpa_chi0_workspace_bytes(grid, cell, q_red, ecut_ha, 2 * n_omega, ...) bytes.
 *   omega_ha[n_omega]: host, finite, any sign; eta_ha > 0 (the broadening; omega = 0, eta = u is the point i u of the
 *   imaginary axis).  Everything else as rpa_chi0_create.
 * On such a handle rpa_chi0_get(i) returns the full complex matrix chi0(omega_i + i eta); rpa_ec_q returns
 * RPA_ERR_UNSUPPORTED (Eq. 2 is an imaginary-axis integral); all add_kpoint variants, reset, the spin setter and the
 * orbital utilities work unchanged.
 */
int rpa_chi0_create_real_axis(rpa_chi0_t **out, const int32_t grid[3], const double cell[9], const double q_red[3],
                              double ecut_ha, int32_t n_omega, const double *omega_ha, double eta_ha,
                              int32_t max_batch_pairs, int32_t max_proj_total, void *workspace, size_t workspace_bytes,
                              void *cuda_stream);

/* Number of G vectors in the sphere. */
int rpa_chi0_ng(const rpa_chi0_t *h, int32_t *ng);

/* g[ng][3] (host, int32): the integer G vectors in the order of every G-indexed array; K2[ng] (host, may be
 * NULL) = |q+G|^2 in bohr^-2. */
int rpa_chi0_gvectors(const rpa_chi0_t *h, int32_t *g, double *K2);

/*
 * Add the transitions of one k-point (Table 1 steps 5, 6, 8, 9, 11):
 *   S_w[G][G'] += kweight * sum_{n < n_occ, m < n_unocc} w_nm(w) n_nm(G) conj(n_nm(G'))   for every omega.
 * All n_occ x n_unocc pairs are included (metallic / smeared occupations allowed, reading A12).
 *   psi_occ   dev cdouble [n_occ][N1][N2][N3]     u_nk;      psi_unocc dev cdouble [n_unocc][N1][N2][N3]  u_m,k+q
 *   eps_occ, f_occ host double [n_occ];  eps_unocc, f_unocc host double [n_unocc]   (Ha; f per spin in [0,1])
 *   n_atoms, n_proj host int32 [n_atoms] (projectors per atom, may differ per atom);  n_atoms = 0: no PAW
 *   P_occ dev cdouble [n_occ][sum n_proj] = <p~^a_i|psi~_nk>;  P_unocc dev cdouble [n_unocc][sum n_proj]
 *   Q dev cdouble, per atom [n_i][n_i][ng] (i, j, G), atoms concatenated; atom-centred (no phase, reading A9)
 *   R_cart host double [n_atoms][3], bohr.
 * Additive and order-independent up to rounding: any split of bands or k-points over calls gives the same chi0.
 */
int rpa_chi0_add_kpoint(rpa_chi0_t *h, double kweight, int32_t n_occ, const void *psi_occ, int32_t n_unocc,
                        const void *psi_unocc, const double *eps_occ, const double *eps_unocc, const double *f_occ,
                        const double *f_unocc, int32_t n_atoms, const int32_t *n_proj, const void *P_occ,
                        const void *P_unocc, const void *Q, const double *R_cart);

/*
 * The same k-point in three steps, for unoccupied orbitals that are still being produced on the handle's stream while the
 * first pair densities are computed -- the paper's own pipeline, where every orbital is expanded from its plane-wave
 * coefficients just before use (Table 1 steps 3-5): uploads and rpa_pw_to_grid calls of later bands go between
 * the steps, and the copies hide under the pair densities of the earlier bands.  Same result as ONE rpa_chi0_add_kpoint
 * call, bit for bit (the same pair densities meet in the same rank-K update).
 *   rpa_chi0_add_kpoint_begin: arguments as rpa_chi0_add_kpoint.  psi_unocc and P_unocc are the full [n_unocc] arrays;
 *     band m of psi_unocc is read by the rpa_chi0_add_kpoint_pairs call that covers m (stream order), P_unocc by
 *     rpa_chi0_add_kpoint_end.  The transitions must fit ONE batch: n_occ n_unocc <= max_batch_pairs of the handle and
 *     n_occ <= 16, else RPA_ERR_UNSUPPORTED and nothing is open (use rpa_chi0_add_kpoint).  Not for q = 0 handles.
 *   rpa_chi0_add_kpoint_pairs(m_begin, m_end): pair densities (S2 + S3) of every occupied band with the unoccupied bands
 *     [m_begin, m_end).  Slices must follow one another: the first starts at 0, each at the end of the one before.
 *   rpa_chi0_add_kpoint_end: PAW correction, weights and the rank-K update of the whole k-point (S4 - S6).
 *     RPA_ERR_INVALID_ARG, nothing added, if the slices did not reach n_unocc.  Closes the k-point in every case.
 * Between begin and end the handle accepts rpa_pw_to_grid, rpa_symmetry_remap, rpa_chi0_get, rpa_ec_q, rpa_chi0_sync;
 * rpa_chi0_add_kpoint* return RPA_ERR_INVALID_ARG.
 */
int rpa_chi0_add_kpoint_begin(rpa_chi0_t *h, double kweight, int32_t n_occ, const void *psi_occ, int32_t n_unocc,
                              const void *psi_unocc, const double *eps_occ, const double *eps_unocc, const double *f_occ,
                              const double *f_unocc, int32_t n_atoms, const int32_t *n_proj, const void *P_occ,
                              const void *P_unocc, const void *Q, const double *R_cart);
int rpa_chi0_add_kpoint_pairs(rpa_chi0_t *h, int32_t m_begin, int32_t m_end);
int rpa_chi0_add_kpoint_end(rpa_chi0_t *h);

/* chi0(i omega_i) = (2/Omega) S_i as a full Hermitian matrix, dev cdouble [ng][ng] row-major (Eq. 3 prefactor,
 * P:L56; spin-paired, reading A3).  Stream-ordered; does not modify the accumulators. */
int rpa_chi0_get(rpa_chi0_t *h, int32_t i_omega, void *chi0_out);

/*
 * E_c(q) = (1/2pi) sum_i wt_i e_i,  e_i = ln det(I - D chi0_i D) + Tr(D chi0_i D),  D = diag(sqrt(v_G))
 * (Eq. 1-2 in the similar Hermitian form, reading A14), by an on-device blocked Cholesky.
 *   v_G host double [ng] (> 0, e.g. 4 pi/|q+G|^2);  ec_ha host double[1];  e_omega host double [n_omega] or NULL.
 * Blocks until done; leaves the accumulators untouched.  Needs omega_wt at create.  RPA_ERR_NOT_PD if a pivot <= 0.
 */
int rpa_ec_q(rpa_chi0_t *h, const double *v_G, double *ec_ha, double *e_omega);

/*
 * The same for the frequencies iw_begin <= i < iw_end only (after a reduce-scatter of the accumulators by
 * frequency every GPU factorises the frequencies it owns; the frequencies are independent terms of Eq. 2):
 *   ec_partial_ha host double[1] = (1/2pi) sum_{i in range} wt_i e_i  -- the sum of the partial values over disjoint
 *   ranges covering [0, n_omega) is E_c(q);  e_omega host double [iw_end - iw_begin] or NULL.
 * Only the accumulators of the range are read, so the others may hold partial sums.  An empty range gives 0.
 * RPA_ERR_INVALID_ARG if the range is not inside [0, n_omega); otherwise as rpa_ec_q.
 */
int rpa_ec_q_range(rpa_chi0_t *h, const double *v_G, int32_t iw_begin, int32_t iw_end, double *ec_partial_ha,
                   double *e_omega);

/*
 * Kernel of the rank-K accumulation S_w += N diag(w) N^H (Eq. 17 / Eq. 20; Table 1 step 11) used by
 * the later rpa_chi0_add_kpoint* calls on this handle.  mode = one RPA_RANK_K_* kind, for RPA_RANK_K_I8 optionally or-ed
 * with RPA_RANK_K_FLAG_* bits.
 *   RPA_RANK_K_FP64_3M (default): FP64 tensor cores (DMMA.8x8x4), complex product by three real contractions
 *       (Re = P1 + P2, Im = P3 - P1 + P2): IEEE double throughout, error ~ K u |n||n'| per element like any FP64 ZHERK.
 *   RPA_RANK_K_FP64_4M: FP64 tensor cores, the plain four-multiplication real view (the reference form of the update).
 *   RPA_RANK_K_I8: for batches with ng >= 768 and >= 1024 transitions, the update is computed on the int8 tensor cores
 *       (tcgen05.mma.kind::i8, s32 accumulators in TMEM) from digit slices of the FP64 operands (Ozaki scheme): every
 *       row g of N, and every row g' of N diag(w) per frequency, is scaled by a power of two 2^-e > its largest
 *       |component| and rounded ONCE to b = 6 + 7 (digits - 1) bits of that scale (digits = 6, 7, 8: b = 41, 48, 55),
 *       the digit products are exact, those below the rounding are dropped, the recombination is FP64.  Error bound per
 *       element, with sL_g = 2^e of row g of N and sR_g' that of row g' of N diag(w), K' = 2 K:
 *           |dS[g][g']| <= (digits + 2) 2^(-7 digits) sL_g sR_g' K'
 *       (first-order: 2 roundings of 2^(-7 digits + 1) / 2 per product plus the digits - 1 dropped pair levels of
 *       2^(-7 digits) each).  It is an ABSOLUTE bound on the scale of the row maxima: an element that is 2^-20 of its row
 *       maximum keeps b - 20 bits, where IEEE double keeps 53 -- narrower than FP64 for rows with a wide dynamic range
 *       (tests/test_gpu_rank_k_i8.py checks this bound element by element on such rows).  Measured on BASELINE configs:
 *       1-5e-14 (digits = 7), 1-3e-12 (6) relative Frobenius distance from the FP64 kernel.  Bitwise reproducible.  Smaller
 *       batches, batches where digits 2 K' 64^2 >= 2^31 (s32 accumulators no longer provably exact: more than 37 448 /
 *       32 768 transitions per batch for 7 / 8 digits), and handles with more than 32 accumulator slots run the default
 *       FP64 kernel.  A NaN or Inf in N or w makes the rows / columns of S it enters non-finite, as in the FP64 kernels.
 *       digits: 6, 7 or 8 (0 = 7); ignored by the FP64 modes.
 *   RPA_RANK_K_FLAG_ALL_BATCHES: take the int8 path for small batches too (tests; it loses time there).
 *   RPA_RANK_K_FLAG_NO_CLUSTER: launch rank_k_i8_kernel without thread-block clusters (no multicast of the row digits).
 * May be called at any time between calls on the handle; RPA_ERR_INVALID_ARG on unknown modes / flags / digits.
 */
#define RPA_RANK_K_FP64_3M 0
#define RPA_RANK_K_FP64_4M 1
#define RPA_RANK_K_I8 2
#define RPA_RANK_K_FLAG_NO_CLUSTER 0x100
#define RPA_RANK_K_FLAG_ALL_BATCHES 0x200
int rpa_chi0_set_rank_k_mode(rpa_chi0_t *h, int32_t mode, int32_t digits);

/* How many rank-K batches have run on the FP64 tensor kernels and on the int8-sliced kernel since create (which path a
 * batch took is otherwise invisible: the results agree to the bound above). */
int rpa_chi0_rank_k_batches(const rpa_chi0_t *h, int64_t *fp64_batches, int64_t *i8_batches);

/* rpa_ec_q factorises the frequencies of a group in n_lanes (1 ... 4, default 2) concurrent shares, each on its own pair
 * of internal streams.  e(omega) does not depend on it (every matrix is factorised by the same kernels in the same order). */
#define RPA_EC_FLAG_WIDE_TILES 0x100 /* or-ed into n_lanes: the updates on the serial chain of the factorisation (strips,
                                       * look-ahead columns) in the 64 x 64 tiles of the big trailing updates instead of
                                       * their own 32 x 32-tile kernel; same results to rounding, for comparison only */
int rpa_chi0_set_ec_lanes(rpa_chi0_t *h, int32_t n_lanes);

/*
 * E_c = sum_q w_q E_c(q): the sum over the irreducible-zone q-points of Eq. 1 (reading A17:
 * rpa_ec_q applies no q weight).  ec_q, q_weights: host double [n_q]; ec_ha: host double[1].  Host arithmetic on the n_q
 * scalars, summed in the order given; n_q = 0 gives 0.
 */
int rpa_total_energy(int32_t n_q, const double *ec_q, const double *q_weights, double *ec_ha);

/*
 * The integrand of Eq. 2 (Table 1 step 12) for ONE matrix, for callers that cannot allocate device
 * memory (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
 *     e = ln det(1 - v^1/2 chi0 v^1/2) + Tr(v^1/2 chi0 v^1/2),
 * the e(omega) of rpa_ec_q, by the same kernels (blocked Cholesky, trailing updates on the FP64 tensor cores) on one
 * stream.  No handle and no workspace: the matrix being factorised, the solved panels and the scalars live in a
 * file-scope device array of the library, RPA_NOALLOC_SCRATCH_BYTES (5 MiB + 2 KiB) per GPU that loads the library,
 * held until the process exits.  The call makes no cudaMalloc / cudaFree and calls no allocating library routine.
 *   chi0:  DEVICE complex128 [ng][ng] row-major as rpa_chi0_get returns it (Hermitian, imaginary axis); only the lower
 *          triangle g >= g' is read; not modified.
 *   ng:    1 ... RPA_NOALLOC_MAX_NG; larger gives RPA_ERR_UNSUPPORTED (use rpa_ec_q), ng < 1 RPA_ERR_INVALID_ARG.
 *   v_G:   DEVICE double [ng], the Coulomb kernel 4 pi / |q+G|^2, every entry finite and > 0 (NOT checked: the call
 *          does not read device memory from the host).
 *   e:     DEVICE double [1]; NaN if a pivot of the factorisation is not positive (where rpa_ec_q returns RPA_ERR_NOT_PD).
 *   cuda_stream: a cudaStream_t (NULL = legacy default stream).  The call only enqueues kernels on it and returns
 *          without synchronising; chi0, v_G and e must stay alive until the stream reaches that point.
 * The first call on a device resolves the device address of the array (cudaGetSymbolAddress) and sets a kernel
 * attribute: make that one outside stream capture, with the device current.  The array is shared by EVERY call in the
 * process on that GPU and keeps the contents of the last one (each call re-initialises what it reads): calls that may
 * overlap on the GPU -- different streams without an ordering between them, or two host threads -- race on it; order
 * them on one stream or with events.  Independent of every rpa_chi0_t handle.
 */
#define RPA_NOALLOC_MAX_NG 512
#define RPA_NOALLOC_SCRATCH_BYTES (RPA_NOALLOC_MAX_NG * RPA_NOALLOC_MAX_NG * 16 + 128 * RPA_NOALLOC_MAX_NG * 16 + 2048)
int rpa_e_omega_noalloc(const void *chi0, int32_t ng, const double *v_G, double *e, void *cuda_stream);

/* Zero the accumulators (start another q with the same sphere). */
int rpa_chi0_reset(rpa_chi0_t *h);

/* Block until all work enqueued on the handle's stream is done; reports asynchronous CUDA errors. */
int rpa_chi0_sync(rpa_chi0_t *h);

/*
 * Per-stage device times (ms, CUDA events on the handle's stream) accumulated by rpa_chi0_add_kpoint while
 * profiling is on: [0] pair product + 2-D FFT, [1] third-axis DFT + sphere gather, [2] PAW, [3] weights,
 * [4] rank-K update (all its kernels), [5] the rank_k_i8_kernel launches alone (a SUBSET of [4], not a further stage; 0
 * when the FP64 tensor kernel ran); launches[6] = kernel launches per stage.  Turning profiling on adds event records only.
 */
int rpa_chi0_set_profiling(rpa_chi0_t *h, int32_t on);
int rpa_chi0_stage_times(rpa_chi0_t *h, double ms[6], int64_t launches[6]);

/* Number of kernel launches enqueued through this handle since it was created. */
int rpa_chi0_launch_count(const rpa_chi0_t *h, int64_t *count);

/*
 * The raw accumulators S[slots][ng][ldS] (dev cdouble, inside the caller's workspace; row pitch ldS >= ng; slots =
 * n_omega, or 2 n_omega on a real-axis handle: Re-weight and Im-weight sums interleaved; only the lower triangle
 * g >= g' is meaningful, the rest is zero) and their size in bytes.  For the multi-GPU sum of per-rank partial
 * chi0 (ranks share nothing until the end of a q): all-reduce this buffer in place on the handle's
 * stream, then call rpa_chi0_get / rpa_ec_q.  The pointer stays valid for the life of the handle.
 */
int rpa_chi0_accumulators(const rpa_chi0_t *h, void **S, size_t *bytes);

/*
 * Table 1 steps 3-4, upstream of rpa_chi0_add_kpoint.
 *
 * rpa_pw_to_grid -- Eq. 10: the cell-periodic part of n_bands pseudo wave functions on the handle's grid
 * from their plane-wave coefficients,
 *     psi_out[b][j1][j2][j3] = sum_Q C[b][Q] exp(+2 pi i (Q1 j1/N1 + Q2 j2/N2 + Q3 j3/N3)),
 * g_pw: host int32 [n_pw][3], the integer reciprocal vectors Q (distinct; any range that fits the scratch);
 * C: dev cdouble [n_bands][n_pw]; psi_out: dev cdouble [n_bands][N1][N2][N3].  No Bloch phase exp(i k.r) is applied
 * (the library works with periodic parts) and no normalisation: (1/N) sum |psi|^2 = sum_Q |C(Q)|^2.
 * Uses the handle's pair-density scratch: stream-ordered with the other calls of the handle.
 * Errors: RPA_ERR_INVALID_ARG (NULL, duplicate Q), RPA_ERR_WORKSPACE / RPA_ERR_UNSUPPORTED (box of the Q too large).
 *
 * rpa_symmetry_remap -- Eq. 11: IBZ -> BZ transformation psi_out(r) = psi_in(T^-1 r), complex conjugated
 * if time_reversal != 0.  M (host int32 [3][3]) is T^-1 in reduced coordinates: the value at fractional coordinates x
 * is taken from M x, i.e. grid index j'_i = sum_k M[i][k] j_k N_i/N_k mod N_i.  psi_in, psi_out: dev cdouble
 * [n_bands][N1][N2][N3], must not alias.  RPA_ERR_UNSUPPORTED if M N_i/N_k is not integer (the operation does not
 * map the grid onto itself).  Fractional translations and the reciprocal-vector shift of a folded-back k are the
 * caller's (reading A5).
 */
int rpa_pw_to_grid(rpa_chi0_t *h, int32_t n_bands, int32_t n_pw, const int32_t *g_pw, const void *C, void *psi_out);
int rpa_symmetry_remap(rpa_chi0_t *h, int32_t n_bands, const int32_t M[9], int32_t time_reversal, const void *psi_in,
                       void *psi_out);

/*
 * Table 1 step 10: the optical limit q -> 0.  A handle created with q_red = (0,0,0)
 * has G = 0 inside its sphere, where Eq. 4 degenerates to delta_nn' and v diverges; the G = 0 element of every pair
 * density is then the perturbative limit of Eq. 13, per unit |q| along a direction qdir,
 *     n_nm(G = 0) = -i qdir . <psi_n| nabla |psi_m> / (eps_m - eps_n)          (0 when eps_m = eps_n),
 * so that with v_G=0 = 4 pi passed to rpa_ec_q the products v^1/2 chi0 v^1/2 are the finite q -> 0 values.
 *
 * rpa_momentum_pw -- Eq. 15 with the plane-wave form of the gradient, Eq. 19 (the paper's GPU
 * reformulation of the CPU code's 13-point stencil):
 *     grad_out[al][n][m] = sum_Q conj(C_occ[n][Q]) i (k_cart + Q B)_al C_unocc[m][Q]
 *                          + sum_a sum_ij conj(P_occ[n][a,i]) Qgrad[a][al][i][j] P_unocc[m][a,j],      al = x, y, z
 * k_cart: host [3] (bohr^-1); g_pw: host int32 [n_pw][3]; C_*: dev cdouble [bands][n_pw], both on the same plane-wave
 * set, sum_Q |C|^2 = 1; Qgrad: dev cdouble, per atom [3][n_i][n_i], atoms concatenated (Eq. 16, computed by the caller
 * from the PAW data sets); n_atoms == 0: no PAW term.  grad_out: dev cdouble [3][n_occ][n_unocc].
 *
 * rpa_chi0_add_kpoint_optical -- rpa_chi0_add_kpoint for a q = 0 handle: same arguments, plus the direction qdir_cart
 * (host [3], normalised by the library) and grad (dev [3][n_occ][n_unocc], e.g. from rpa_momentum_pw).  On a q = 0
 * handle the plain rpa_chi0_add_kpoint returns RPA_ERR_UNSUPPORTED, on a q != 0 handle this call returns
 * RPA_ERR_INVALID_ARG.
 */
int rpa_momentum_pw(rpa_chi0_t *h, const double k_cart[3], int32_t n_pw, const int32_t *g_pw, int32_t n_occ, const void *C_occ,
                    int32_t n_unocc, const void *C_unocc, int32_t n_atoms, const int32_t *n_proj, const void *P_occ,
                    const void *P_unocc, const void *Qgrad, void *grad_out);
int rpa_chi0_add_kpoint_optical(rpa_chi0_t *h, double kweight, int32_t n_occ, const void *psi_occ, int32_t n_unocc,
                                const void *psi_unocc, const double *eps_occ, const double *eps_unocc, const double *f_occ,
                                const double *f_unocc, int32_t n_atoms, const int32_t *n_proj, const void *P_occ,
                                const void *P_unocc, const void *Q, const double *R_cart, const double qdir_cart[3],
                                const void *grad);

/*
 * Spin-polarised systems ("the spin index sigma is implicitly contained").  The prefactor
 * of chi0 = (s/Omega) S is s = 2 by default (spin-paired bands, reading A3).  With s = 1 the caller adds the bands of
 * each spin channel with their own rpa_chi0_add_kpoint calls (f in [0,1] per channel); rpa_chi0_get and rpa_ec_q then
 * use 1/Omega.  s must be 1 or 2; it may be changed at any time (it scales the read-out, not the accumulators).
 */
int rpa_chi0_set_spin_degeneracy(rpa_chi0_t *h, int32_t s);

void rpa_chi0_destroy(rpa_chi0_t *h);

/* Thread-local message of the last error on this thread (static storage, never NULL). */
const char *rpa_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* RPA_CHI0_H */
