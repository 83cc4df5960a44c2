// pd_zy_kernel -- pair product + z and y transforms of the pruned 3-D FFT (Table 1 step 5; Eq. 12,
// P:L104-106) for planes that fit one CTA, written for a low instruction count per grid point: every loop is
// unrolled at compile time, all shared-memory addresses are a per-thread base plus constants.
//
// Both axes use the same two-level split N = NA * NB:
//   pass A  (full)    A_j[k1] = sum_s x[j + NB s] W_NA^(s k1)            one radix-NA butterfly in registers
//   pass B  (pruned)  X[f]    = sum_j W_N^(j f) A_j[f mod NA]            direct NB-term sum, only for f in the box
// so the work after the butterfly is proportional to the number of frequencies kept (ng3 of N3, ng2 of N2).
//
// z axis: a warp owns LPW whole lines (NB3 lanes per line): pass A -> padded exchange buffer of the warp -> pass B
// needs __syncwarp only, no block barrier.  u_m is prefetched into registers TWO iterations ahead (two register
// buffers used alternately; plain 16-byte loads, 128 contiguous bytes per line and instruction), which covers the
// HBM latency with 8 warps per SM.  The chunk of u_n is reused for the G pairs (same occupied band) a CTA
// transforms together, so it costs 1/G global loads per point; it lives in thread-private shared-memory slots
// (cp.async, conflict-free [element][thread] layout) to leave the registers to the second prefetch buffer.
// y axis: the ng3 * G surviving columns: pass A in place in shared memory, pass B writes I[pair][j1][g2i][g3i]
// (coalesced: consecutive threads -> consecutive g3i).
#pragma once
#include "fft.cuh"

#define PDZY_MAXK1 4   // k1 values per z pass-B thread: ceil(NA3 / NB3)

// cos / sin of 2 pi num / den as compile-time constants (Taylor series in long double after reduction to
// [-pi, pi]; error < 1e-18): the pruned pass-B sums below then multiply by immediates / constant-bank operands.
__host__ __device__ constexpr long double pdzy_angle(int num, int den) {
    int r = num % den;
    if (r < 0) r += den;
    if (2 * r > den) r -= den;
    return 2.0L * 3.14159265358979323846264338327950288L * (long double)r / (long double)den;
}
__host__ __device__ constexpr double pdzy_cos(int num, int den) {
    const long double x = pdzy_angle(num, den);
    long double term = 1.0L, sum = 1.0L;
    for (int k = 1; k <= 24; k++) {
        term *= -x * x / (long double)((2 * k - 1) * (2 * k));
        sum += term;
    }
    return (double)sum;
}
__host__ __device__ constexpr double pdzy_sin(int num, int den) {
    const long double x = pdzy_angle(num, den);
    long double term = x, sum = x;
    for (int k = 1; k <= 24; k++) {
        term *= -x * x / (long double)((2 * k) * (2 * k + 1));
        sum += term;
    }
    return (double)sum;
}

// z pass B: with N = NA NB and x[j] = W_N^(j k1) A_j[k1], the frequencies f = k1 + NA d kept by the box are
//   out[d - DLO] = sum_{j < NB} W_NB^(j d) x[j],   d = DLO .. DHI   (a pruned NB-point DFT).
// For even NB halves first (W_NB^((j + NB/2) d) = (-1)^d W_NB^(j d)): e = x_lo + x_hi feeds even d, f = x_lo - x_hi odd d; then
// +d and -d share the cosine and sine sums P = sum cos(2 pi j d / NB) s_j, Q = sum sin(2 pi j d / NB) s_j:
//   out[+d] = P - i Q,  out[-d] = P + i Q.
template <int NB, int DLO, int DHI>
struct PrunedDft {
    static_assert(DLO <= 0 && DHI >= 0, "pruned DFT");
    static constexpr bool EVEN = (NB % 2 == 0);
    static constexpr int H = EVEN ? NB / 2 : NB;   // terms per sum
    static constexpr int ADMAX = (-DLO > DHI) ? -DLO : DHI;
    template <int AD, int J>
    __device__ __forceinline__ static void acc(const cd *s, cd &Pv, cd &Qv) {
        if constexpr (J < H) {
            constexpr double c = pdzy_cos(J * AD, NB), sn = pdzy_sin(J * AD, NB);
            if constexpr (J == 0) {
                Pv = s[0];
                Qv = make_double2(0.0, 0.0);
            } else {
                Pv = make_double2(fma(c, s[J].x, Pv.x), fma(c, s[J].y, Pv.y));
                Qv = make_double2(fma(sn, s[J].x, Qv.x), fma(sn, s[J].y, Qv.y));
            }
            acc<AD, J + 1>(s, Pv, Qv);
        }
    }
    template <int AD>
    __device__ __forceinline__ static void level(const cd *e, const cd *f, cd *out) {
        if constexpr (AD <= ADMAX) {
            const cd *s = (AD % 2 == 0) ? e : f;
            if constexpr (AD == 0) {
                cd t = s[0];
#pragma unroll
                for (int j = 1; j < H; j++) t = h_add(t, s[j]);
                out[-DLO] = t;
            } else {
                cd Pv, Qv;
                acc<AD, 0>(s, Pv, Qv);
                if constexpr (AD <= DHI) out[AD - DLO] = make_double2(Pv.x + Qv.y, Pv.y - Qv.x);
                if constexpr (-AD >= DLO) out[-AD - DLO] = make_double2(Pv.x - Qv.y, Pv.y + Qv.x);
            }
            level<AD + 1>(e, f, out);
        }
    }
    __device__ __forceinline__ static void run(const cd *x, cd *out) {
        if constexpr (EVEN) {
            cd e[H], f[H];
#pragma unroll
            for (int j = 0; j < H; j++) {
                e[j] = h_add(x[j], x[j + H]);
                f[j] = h_sub(x[j], x[j + H]);
            }
            level<0>(e, f, out);
        } else {
            level<0>(x, x, out);
        }
    }
};

struct PdZyParams {
    const cd *psi_occ, *psi_unocc;  // [band][N1][N2][N3]
    cd *I;                          // [pair - p_begin][N1][ncols]: only the (g2, g3) columns that hold sphere points
    const int32_t *coltab;          // [ncols]: (g2i << 16) | g3i of column c, ascending in g2i ng3 + g3i
    const int32_t *rowtab;          // [ng2 + 1]: first column of every g2i
    int ncols;
    const cd *tw3, *tw2;            // exp(-2 pi i t/N3), exp(-2 pi i t/N2)
    int N1;
    int n0, mlen, m0;               // pair p of the batch -> band n = n0 + p / mlen, m = m0 + p % mlen
    int p_begin, p_count;           // pairs of the batch handled by this launch
    int n_units;                    // groups of <= G consecutive pairs with the same occupied band
    // closed-form unit -> pair map (pdzy_plan_units): the launch's first row (pairs of one occupied band) may start in its
    // middle and holds nu0 units; every later row starts a fresh unit and holds upr = ceil(mlen / G) units, the last one
    // possibly cut short by the end of the launch.  Divisions by N1 and upr are multiplications by 2^64 / d rounded up.
    int row0, nu0, upr;
    unsigned long long magic_n1, magic_upr;
    int g2min, ng2, g3min, ng3;
};

template <int N3, int NA3, int DLO, int DHI, int N2, int NA2, int NW, int LPW, int G>
struct PdZy {
    static constexpr int NB3 = N3 / NA3, NB2 = N2 / NA2;
    static constexpr int K1PT = (NA3 + NB3 - 1) / NB3;
    // exchange line of the z stage: element (k1, j) at k1 XP + j, lines XLINE apart (units of 16 bytes).  Pitches found by
    // enumerating the quarter-warp bank groups of the pass-A stores (k1 fixed) and pass-B loads (j fixed) of this lane
    // layout: conflict-free for NB3 = 2, 3, 8, 16, 10 % over the minimum for NB3 = 14
    static constexpr int XP = NB3 == 2 ? 3 : NB3 == 3 ? 9 : NB3 == 14 ? 17 : NB3 + ((NB3 & 1) ? 0 : 1);
        // NB3 = 4 (two lines per quarter-warp): stores hit lw XLINE + j, loads lw XLINE + j XP: XP = 5 and XLINE = 4 mod 8 make
    // both sets {0..7} (XLINE = NA3 XP = 30 gave two-way conflicts on both: 27 % of the kernel's wavefronts on configs[2])
    static constexpr int XLINE = NB3 == 2 ? 26 : NB3 == 3 ? 75 : NB3 == 14 ? 206 : NB3 == 4 ? ((NA3 - 1) * XP + NB3 + 7) / 8 * 8 + 4 : NA3 * XP;
    static_assert(XLINE >= (NA3 - 1) * XP + NB3, "exchange line too short");
    static constexpr int ROWS = NW * LPW;                 // z lines per chunk
    static constexpr int NCH = (N2 + ROWS - 1) / ROWS;
    static constexpr int NTH = NW * 32;
    static_assert(N3 % NA3 == 0 && N2 % NA2 == 0, "split");
    static_assert(LPW * NB3 <= 32, "lanes");
    static_assert(K1PT <= PDZY_MAXK1, "k1 per thread");

    // shared memory (cd): tw2[N2] | X[NW][LPW][XLINE] | UN[NA3][NTH] | Y[N2][G * ng3] ; then int32 otab[ng2 * ng3]
    static size_t smem_bytes(int ng2, int ng3) {
        return ((size_t)N2 + (size_t)NW * LPW * XLINE + (size_t)NA3 * NTH + (size_t)N2 * G * ng3) * sizeof(cd) +
               (size_t)ng2 * ng3 * sizeof(int32_t);
    }
    static constexpr int ND = DHI - DLO + 1;
    static_assert(NA3 * ND <= N3, "kept frequencies must be distinct modulo N3");
    // the z pass B keeps g = k1 + NA3 d, d = DLO .. DHI: the box must lie inside [NA3 DLO, NA3 (DHI + 1))
    static bool box_ok(int g3min, int ng3) { return g3min >= NA3 * DLO && g3min + ng3 <= NA3 * (DHI + 1); }
};

// x / d for any 0 <= x < 2^31, d >= 1 as the high half of a 64 x 64 multiplication: magic = floor((2^64 - 1) / d) + 1, so
// magic d = 2^64 + e with 0 < e <= d and x magic / 2^64 = x / d + x e / (d 2^64), whose excess stays below 1 / d.
// d = 1 has no 64-bit magic: it is encoded as 0.
static inline unsigned long long pdzy_magic(int d) { return d <= 1 ? 0ull : ~0ull / (unsigned long long)d + 1ull; }
__host__ __device__ __forceinline__ int pdzy_fastdiv(int x, unsigned long long magic) {
#ifdef __CUDA_ARCH__
    return magic ? (int)__umul64hi((unsigned long long)(unsigned)x, magic) : x;
#else   // the host copy exists for tests/host/unit_map_check.cu
    return magic ? (int)(((unsigned __int128)(unsigned)x * magic) >> 64) : x;
#endif
}

// unit u of the launch -> first pair p (relative to the batch) and the number of pairs cnt <= G, all in one row r.
template <int G>
__host__ __device__ __forceinline__ void pdzy_unit(const PdZyParams &P, int u, int &p, int &cnt, int &r) {
    if (u < P.nu0) {
        r = P.row0;
        p = P.p_begin + u * G;
    } else {
        const int u2 = u - P.nu0, q = pdzy_fastdiv(u2, P.magic_upr);
        r = P.row0 + 1 + q;
        p = r * P.mlen + (u2 - q * P.upr) * G;
    }
    const int rest = ((r + 1) * P.mlen < P.p_begin + P.p_count ? (r + 1) * P.mlen : P.p_begin + P.p_count) - p;
    cnt = rest < G ? rest : G;
}

// host: fills n_units, row0, nu0, upr and the division constants of a launch over pairs [p_begin, p_begin + p_count)
template <class Params>
static inline void pdzy_plan_units(Params &P, int G) {
    const int p_end = P.p_begin + P.p_count;
    P.row0 = P.p_begin / P.mlen;
    const int first_end = std::min((P.row0 + 1) * P.mlen, p_end);
    P.nu0 = (first_end - P.p_begin + G - 1) / G;
    P.upr = (P.mlen + G - 1) / G;
    int n = P.nu0;
    for (int p = first_end; p < p_end; p += P.mlen) n += (std::min(p + P.mlen, p_end) - p + G - 1) / G;
    P.n_units = n;
    P.magic_n1 = pdzy_magic(P.N1);
    P.magic_upr = pdzy_magic(P.upr);
}


__device__ __forceinline__ void pdzy_cp_async16(void *dst_smem, const void *src_gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void pdzy_cp_async_wait() {
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
}

// position of a CTA in its sequence of z iterations: work item w = u N1 + j1 (unit u: pairs p0 .. p0 + cnt - 1 of
// occupied band n, first unoccupied band m; plane j1), chunk c of the plane, pair g of the unit.  The grid is 1-D
// and persistent (CTAs = resident slots of the GPU): CTA b takes items b, b + gridDim.x, ...
struct PdZyCursor {
    int w, p0, cnt, n, m, c, g, j1;
};

// YROW: y pass B with one output row per thread and its twiddles in registers (else tasks dealt round-robin with the
// twiddles read from shared memory); measured better for the 60- and 48-row planes, worse for 24 and 40
template <int N3, int NA3, int DLO, int DHI, int N2, int NA2, int NW, int LPW, int G, int MINB, bool YROW = false>
__global__ void __launch_bounds__(NW * 32, MINB) pd_zy_kernel(const __grid_constant__ PdZyParams P) {
    using C = PdZy<N3, NA3, DLO, DHI, N2, NA2, NW, LPW, G>;
    constexpr int ND = C::ND;
    constexpr int NB3 = C::NB3, NB2 = C::NB2, K1PT = C::K1PT, XP = C::XP, XLINE = C::XLINE, ROWS = C::ROWS, NCH = C::NCH,
                  NTH = C::NTH;
    extern __shared__ __align__(16) unsigned char pd_smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int ng2 = P.ng2, ng3 = P.ng3, nb2 = P.ncols;   // nb2: columns kept (pitch of I), <= ng2 ng3
    cd *tw2s = reinterpret_cast<cd *>(pd_smem);
    cd *X = tw2s + N2;
    cd *UN = X + NW * LPW * XLINE;
    cd *Y = UN + NA3 * NTH;
    int32_t *otab = reinterpret_cast<int32_t *>(Y + (size_t)N2 * G * ng3);
    for (int i = tid; i < N2; i += NTH) tw2s[i] = P.tw2[i];
    for (int i = tid; i < nb2; i += NTH) otab[i] = P.coltab[i];

    // ---- this thread's z role: line lw of the warp, butterfly / pass-B slot j ------------------------------------
    const int lw = lane / NB3, j = lane - lw * NB3;
    const bool zact = lw < LPW;
    cd *Xl = X + (warp * LPW + (zact ? lw : 0)) * XLINE;
    cd *uns = UN + tid;   // this thread's u_n elements: uns[t * NTH]
    // pass B: k1 = j + a NB3 keeps g = k1 + NA3 d, d = DLO .. DHI (box index oi, -1 outside); twiddles W_N3^(jj k1)
    cd twb[K1PT][NB3];
    int oi[K1PT][ND];
#pragma unroll
    for (int a = 0; a < K1PT; a++) {
        const int k1 = j + a * NB3;
#pragma unroll
        for (int d = 0; d < ND; d++) {
            const int i = k1 + NA3 * (d + DLO) - P.g3min;
            oi[a][d] = (k1 < NA3 && i >= 0 && i < ng3) ? i : -1;
        }
#pragma unroll
        for (int jj = 0; jj < NB3; jj++) twb[a][jj] = P.tw3[(jj * (k1 < NA3 ? k1 : 0)) % N3];
    }

    constexpr int plane = N2 * N3;
    const size_t vol = (size_t)plane * P.N1;
    // element offset of this thread's first input inside a plane, chunk 0: row (warp LPW + lw), column j
    const int row_in_chunk = warp * LPW + lw;
    const int off0 = row_in_chunk * N3 + j;
    const int n_items = P.n_units * P.N1;

    auto decode = [&](PdZyCursor &k) {   // k.w set; fills the other fields (cnt = 0 past the end)
        k.c = 0;
        k.g = 0;
        k.cnt = 0;
        if (k.w < n_items) {
            const int u = pdzy_fastdiv(k.w, P.magic_n1);
            int r;
            k.j1 = k.w - u * P.N1;
            pdzy_unit<G>(P, u, k.p0, k.cnt, r);
            k.n = P.n0 + r;
            k.m = P.m0 + k.p0 - r * P.mlen;
        }
    };
    auto advance = [&](PdZyCursor &k) {
        if (++k.g >= k.cnt) {
            k.g = 0;
            if (++k.c == NCH) {
                k.w += gridDim.x;
                decode(k);
            }
        }
    };
    auto load_m = [&](cd (&nx)[NA3], const PdZyCursor &k) {
        if (k.cnt > 0 && zact && k.c * ROWS + row_in_chunk < N2) {
            const cd *s = P.psi_unocc + (size_t)(k.m + k.g) * vol + (k.j1 * plane + k.c * ROWS * N3 + off0);
#pragma unroll
            for (int t = 0; t < NA3; t++) nx[t] = __ldcs(s + t * NB3);  // streamed once
        }
    };
    auto load_n = [&](const PdZyCursor &k) {   // u_n chunk of the cursor -> this thread's shared-memory slots
        if (k.cnt > 0 && zact && k.c * ROWS + row_in_chunk < N2) {
            const cd *s = P.psi_occ + (size_t)k.n * vol + (k.j1 * plane + k.c * ROWS * N3 + off0);
#pragma unroll
            for (int t = 0; t < NA3; t++) pdzy_cp_async16(uns + t * NTH, s + t * NB3);
        }
    };

    PdZyCursor cur, pf;
    cur.w = blockIdx.x;
    cur.p0 = cur.n = cur.m = cur.j1 = 0;
    decode(cur);
    pf = cur;
    cd nxA[NA3], nxB[NA3];
    load_n(cur);
    load_m(nxA, pf);
    if (pf.cnt > 0) advance(pf);
    load_m(nxB, pf);
    if (pf.cnt > 0) advance(pf);
    // y pass-B start position of this thread: task t = tid -> (pair g, r = o ng3 + col)
    const int yb_g0 = tid / nb2, yb_r0 = tid - yb_g0 * nb2;
    // YROW: output row o = tid / tpo (tpo threads per row), first column tid % tpo; the row's frequency f, its source
    // rows NB2 (f mod NA2) + j2 and its twiddles W_N2^(j2 f) never change
    const int yb_tpo = max(1, NTH / ng2);
    const int yb_o = (tid / yb_tpo < ng2) ? tid / yb_tpo : -1, yb_c0 = tid % yb_tpo;
    int yb_row = 0, yb_rs = 0, yb_rc = 0;   // YROW: source row block, first kept column of the row, kept columns in it
    cd ytw[(YROW && NB2 > 1) ? NB2 - 1 : 1];
    if constexpr (YROW) {
        if (yb_o >= 0) {
            yb_rs = P.rowtab[yb_o];
            yb_rc = P.rowtab[yb_o + 1] - yb_rs;
        }
        int f = P.g2min + (yb_o >= 0 ? yb_o : 0);
        f %= N2;
        if (f < 0) f += N2;
        yb_row = NB2 * (f % NA2);
#pragma unroll
        for (int j2 = 1; j2 < NB2; j2++) ytw[j2 - 1] = P.tw2[(j2 * f) % N2];
    }
    __syncthreads();

    // one z iteration (chunk c of pair g of the unit) on the inputs in nx; refills nx for two iterations later
    auto step = [&](cd (&nx)[NA3]) {
        const int c = cur.c, g = cur.g, cnt = cur.cnt, p0 = cur.p0, j1 = cur.j1;
        const int row = c * ROWS + row_in_chunk;
        const bool act = zact && row < N2;
        const int pitch = cnt * ng3;   // Y row pitch of this unit: [row][g][g3i]
        if (g == 0) pdzy_cp_async_wait();   // u_n of this chunk has landed in this thread's slots
        cd v[NA3];
#pragma unroll
        for (int t = 0; t < NA3; t++) v[t] = cmulc(uns[t * NTH], nx[t]);
        load_m(nx, pf);
        if (pf.cnt > 0) advance(pf);
        advance(cur);
        if (g + 1 == cnt) load_n(cur);   // next chunk's u_n: the slots have just been read (in-order LSU)
        if (act) {
            Bfly<NA3>::run(v);
#pragma unroll
            for (int t = 0; t < NA3; t++) Xl[t * XP + j] = v[t];
        }
        __syncwarp();
        if (act) {
            cd *yrow = Y + (size_t)row * pitch + g * ng3;
#pragma unroll
            for (int a = 0; a < K1PT; a++) {
                if (j + a * NB3 < NA3) {
                    cd B[NB3];
                    B[0] = Xl[(j + a * NB3) * XP];
#pragma unroll
                    for (int jj = 1; jj < NB3; jj++) B[jj] = h_mul(twb[a][jj], Xl[(j + a * NB3) * XP + jj]);
                    cd o[ND];
                    PrunedDft<NB3, DLO, DHI>::run(B, o);
#pragma unroll
                    for (int d = 0; d < ND; d++)
                        if (oi[a][d] >= 0) yrow[oi[a][d]] = o[d];
                }
            }
        }
        __syncwarp();
        if (c != NCH - 1 || g + 1 != cnt) return;

        // ---- last z iteration of the unit: y axis on its cnt * ng3 columns ------------------------------------------
        __syncthreads();
        {   // pass A in place: x = j2 pitch + (g, g3i); inputs at rows j2 + NB2 s, outputs k1 at the same rows
            const int ntask = NB2 * pitch;
            for (int x = tid; x < ntask; x += NTH) {
                cd w[NA2];
#pragma unroll
                for (int s = 0; s < NA2; s++) w[s] = Y[x + s * ntask];
                Bfly<NA2>::run(w);
#pragma unroll
                for (int s = 0; s < NA2; s++) Y[x + s * ntask] = w[s];
            }
        }
        __syncthreads();
        if constexpr (YROW) {   // pass B, this thread's output row: its kept columns, yb_tpo threads per row, for every pair
            if (yb_o >= 0) {
                cd *Io = P.I + ((size_t)(p0 - P.p_begin) * P.N1 + j1) * nb2 + yb_rs;
                const cd *src = Y + (size_t)yb_row * pitch;
                // (pair, kept column of the row) flattened, yb_tpo threads per row
                int gg = 0, idx = yb_c0;
                while (idx >= yb_rc && gg < cnt) { idx -= yb_rc; gg++; }
                while (gg < cnt) {
                    const int col = otab[yb_rs + idx] & 0xffff;
                    const cd *sp = src + gg * ng3 + col;
                    cd acc = sp[0];
#pragma unroll
                    for (int j2 = 1; j2 < NB2; j2++) acc = cfma(ytw[j2 - 1], sp[j2 * pitch], acc);
                    Io[(size_t)gg * P.N1 * nb2 + idx] = acc;
                    idx += yb_tpo;
                    while (idx >= yb_rc && gg < cnt) { idx -= yb_rc; gg++; }
                }
            }
        } else {   // pass B: out[g][o][g3i] = sum_j2 W_N2^(j2 f) A[j2 + NB2 (f mod NA2)][g][g3i]
            int gg = yb_g0, r = yb_r0;
            cd *Io = P.I + ((size_t)(p0 - P.p_begin) * P.N1 + j1) * nb2;
            while (gg < cnt) {
                const int oc = otab[r];
                const int o = oc >> 16, col = oc & 0xffff;
                int f = P.g2min + o;
                if (f < 0) f += N2;
                const int k1 = f % NA2;
                const cd *src = Y + (size_t)(NB2 * k1) * pitch + gg * ng3 + col;
                cd acc = src[0];
                int ti = 0;
#pragma unroll
                for (int j2 = 1; j2 < NB2; j2++) {
                    ti += f;
                    if (ti >= N2) ti -= N2;
                    acc = cfma(tw2s[ti], src[j2 * pitch], acc);
                }
                Io[(size_t)gg * P.N1 * nb2 + r] = acc;
                r += NTH;
                while (r >= nb2) { r -= nb2; gg++; }
            }
        }
        __syncthreads();   // Y is rewritten by the next unit's z stage
    };

    while (cur.cnt > 0) {
        step(nxA);
        if (cur.cnt == 0) break;
        step(nxB);
    }
}

typedef void (*PdZyKernel)(const PdZyParams);
