// Mixed-radix Stockham FFT building blocks (radices 2,3,4,5,6,7,8), forward sign exp(-2 pi i jk/N).
// Used by the pair-density kernels (Eq. 12; Table 1 step 5).  The butterflies and the
// per-pass index arithmetic are __host__ __device__ so they can be exercised on the build box without a GPU.
#pragma once
#include "common.cuh"

#define FFT_MAX_PASSES 10

struct FftPlan {
    int n;                     // line length
    int npass;                 // number of Stockham passes
    int radix[FFT_MAX_PASSES]; // product = n
};

#ifndef __CUDACC__
#define HD
#else
#define HD __host__ __device__ __forceinline__
#endif

HD cd h_add(cd a, cd b) { return make_double2(a.x + b.x, a.y + b.y); }
HD cd h_sub(cd a, cd b) { return make_double2(a.x - b.x, a.y - b.y); }
HD cd h_mul(cd a, cd b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
HD cd h_mni(cd a) { return make_double2(a.y, -a.x); }  // -i a
HD cd h_mpi(cd a) { return make_double2(-a.y, a.x); }  // +i a
HD cd h_scale(double s, cd a) { return make_double2(s * a.x, s * a.y); }

template <int R>
struct Bfly;

template <>
struct Bfly<2> {
    HD static void run(cd *v) {
        cd a = v[0], b = v[1];
        v[0] = h_add(a, b);
        v[1] = h_sub(a, b);
    }
};

template <>
struct Bfly<4> {
    HD static void run(cd *v) {
        cd s02 = h_add(v[0], v[2]), d02 = h_sub(v[0], v[2]);
        cd s13 = h_add(v[1], v[3]), d13 = h_sub(v[1], v[3]);
        v[0] = h_add(s02, s13);
        v[2] = h_sub(s02, s13);
        v[1] = h_add(d02, h_mni(d13));  // d02 - i d13
        v[3] = h_add(d02, h_mpi(d13));  // d02 + i d13
    }
};

template <>
struct Bfly<8> {
    HD static void run(cd *v) {
        const double h = 0.70710678118654752440;
        cd e[4] = {v[0], v[2], v[4], v[6]};
        cd o[4] = {v[1], v[3], v[5], v[7]};
        Bfly<4>::run(e);
        Bfly<4>::run(o);
        // W8^k o_k
        cd t1 = make_double2(h * (o[1].x + o[1].y), h * (o[1].y - o[1].x));   // (1-i)/sqrt2 * o1
        cd t2 = h_mni(o[2]);                                                   // -i o2
        cd t3 = make_double2(h * (o[3].y - o[3].x), -h * (o[3].x + o[3].y));  // (-1-i)/sqrt2 * o3
        v[0] = h_add(e[0], o[0]);
        v[4] = h_sub(e[0], o[0]);
        v[1] = h_add(e[1], t1);
        v[5] = h_sub(e[1], t1);
        v[2] = h_add(e[2], t2);
        v[6] = h_sub(e[2], t2);
        v[3] = h_add(e[3], t3);
        v[7] = h_sub(e[3], t3);
    }
};

template <>
struct Bfly<3> {
    HD static void run(cd *v) {
        const double s = 0.86602540378443864676;  // sin(2 pi/3)
        cd t1 = h_add(v[1], v[2]);
        cd t2 = make_double2(v[0].x - 0.5 * t1.x, v[0].y - 0.5 * t1.y);
        cd t3 = h_scale(s, h_sub(v[1], v[2]));
        v[0] = h_add(v[0], t1);
        v[1] = h_add(t2, h_mni(t3));
        v[2] = h_add(t2, h_mpi(t3));
    }
};

template <>
struct Bfly<5> {
    HD static void run(cd *v) {
        const double c1 = 0.30901699437494742410, c2 = -0.80901699437494742410;  // cos(2pi/5), cos(4pi/5)
        const double s1 = 0.95105651629515357212, s2 = 0.58778525229247312917;   // sin(2pi/5), sin(4pi/5)
        cd a = h_add(v[1], v[4]), b = h_add(v[2], v[3]);
        cd c = h_sub(v[1], v[4]), d = h_sub(v[2], v[3]);
        cd m1 = make_double2(v[0].x + c1 * a.x + c2 * b.x, v[0].y + c1 * a.y + c2 * b.y);
        cd m2 = make_double2(v[0].x + c2 * a.x + c1 * b.x, v[0].y + c2 * a.y + c1 * b.y);
        cd n1 = make_double2(s1 * c.x + s2 * d.x, s1 * c.y + s2 * d.y);
        cd n2 = make_double2(s2 * c.x - s1 * d.x, s2 * c.y - s1 * d.y);
        v[0] = h_add(v[0], h_add(a, b));
        v[1] = h_add(m1, h_mni(n1));
        v[4] = h_add(m1, h_mpi(n1));
        v[2] = h_add(m2, h_mni(n2));
        v[3] = h_add(m2, h_mpi(n2));
    }
};

template <>
struct Bfly<7> {
    HD static void run(cd *v) {
        // cos/sin(2 pi k/7), k = 1..3
        const double c1 = 0.62348980185873353053, c2 = -0.22252093395631440429, c3 = -0.90096886790241912624;
        const double s1 = 0.78183148246802980871, s2 = 0.97492791218182360702, s3 = 0.43388373911755812048;
        cd a1 = h_add(v[1], v[6]), a2 = h_add(v[2], v[5]), a3 = h_add(v[3], v[4]);
        cd d1 = h_sub(v[1], v[6]), d2 = h_sub(v[2], v[5]), d3 = h_sub(v[3], v[4]);
        cd v0 = v[0];
        // y_f = v0 + sum_k cos(2pi f k/7) a_k - i sum_k sin(2pi f k/7) d_k ; y_{7-f} with +i
        cd m1 = make_double2(v0.x + c1 * a1.x + c2 * a2.x + c3 * a3.x, v0.y + c1 * a1.y + c2 * a2.y + c3 * a3.y);
        cd m2 = make_double2(v0.x + c2 * a1.x + c3 * a2.x + c1 * a3.x, v0.y + c2 * a1.y + c3 * a2.y + c1 * a3.y);
        cd m3 = make_double2(v0.x + c3 * a1.x + c1 * a2.x + c2 * a3.x, v0.y + c3 * a1.y + c1 * a2.y + c2 * a3.y);
        // f=1: sin(k); f=2: sin(2k): s2, s4=-s3, s6=-s1 ; f=3: sin(3k): s3, s6=-s1, s9=s2
        cd n1 = make_double2(s1 * d1.x + s2 * d2.x + s3 * d3.x, s1 * d1.y + s2 * d2.y + s3 * d3.y);
        cd n2 = make_double2(s2 * d1.x - s3 * d2.x - s1 * d3.x, s2 * d1.y - s3 * d2.y - s1 * d3.y);
        cd n3 = make_double2(s3 * d1.x - s1 * d2.x + s2 * d3.x, s3 * d1.y - s1 * d2.y + s2 * d3.y);
        v[0] = h_add(v0, h_add(a1, h_add(a2, a3)));
        v[1] = h_add(m1, h_mni(n1));
        v[6] = h_add(m1, h_mpi(n1));
        v[2] = h_add(m2, h_mni(n2));
        v[5] = h_add(m2, h_mpi(n2));
        v[3] = h_add(m3, h_mni(n3));
        v[4] = h_add(m3, h_mpi(n3));
    }
};

template <>
struct Bfly<6> {
    // 6 = 2 x 3 Cooley-Tukey in registers: j = 2 j1 + j0, k = k0 + 3 k1
    HD static void run(cd *v) {
        const double s = 0.86602540378443864676;
        cd e[3] = {v[0], v[2], v[4]};
        cd o[3] = {v[1], v[3], v[5]};
        Bfly<3>::run(e);
        Bfly<3>::run(o);
        // W6^1 = 1/2 - i s ; W6^2 = -1/2 - i s
        cd t1 = make_double2(0.5 * o[1].x + s * o[1].y, 0.5 * o[1].y - s * o[1].x);
        cd t2 = make_double2(-0.5 * o[2].x + s * o[2].y, -0.5 * o[2].y - s * o[2].x);
        v[0] = h_add(e[0], o[0]);
        v[3] = h_sub(e[0], o[0]);
        v[1] = h_add(e[1], t1);
        v[4] = h_sub(e[1], t1);
        v[2] = h_add(e[2], t2);
        v[5] = h_sub(e[2], t2);
    }
};

template <>
struct Bfly<12> {
    // 12 = 4 x 3 Cooley-Tukey in registers: j = 3 j1 + j2 (j1 < 4, j2 < 3), k = k1 + 4 k2:
    //   X[k1 + 4 k2] = sum_j2 W3^(j2 k2) W12^(j2 k1) sum_j1 v[3 j1 + j2] W4^(j1 k1)
    HD static void run(cd *v) {
        const double c = 0.86602540378443864676;  // cos(pi/6) = sin(pi/3)
        cd e[3][4];
#pragma unroll
        for (int j2 = 0; j2 < 3; j2++) {
            e[j2][0] = v[j2]; e[j2][1] = v[j2 + 3]; e[j2][2] = v[j2 + 6]; e[j2][3] = v[j2 + 9];
            Bfly<4>::run(e[j2]);
        }
        // W12^(j2 k1): W12 = c - i/2, W12^2 = 1/2 - i c, W12^3 = -i, W12^4 = -1/2 - i c, W12^6 = -1
        cd a;
        a = e[1][1]; e[1][1] = make_double2(c * a.x + 0.5 * a.y, c * a.y - 0.5 * a.x);
        a = e[1][2]; e[1][2] = make_double2(0.5 * a.x + c * a.y, 0.5 * a.y - c * a.x);
        e[1][3] = h_mni(e[1][3]);
        a = e[2][1]; e[2][1] = make_double2(0.5 * a.x + c * a.y, 0.5 * a.y - c * a.x);
        a = e[2][2]; e[2][2] = make_double2(-0.5 * a.x + c * a.y, -0.5 * a.y - c * a.x);
        e[2][3] = make_double2(-e[2][3].x, -e[2][3].y);
#pragma unroll
        for (int k1 = 0; k1 < 4; k1++) {
            cd t[3] = {e[0][k1], e[1][k1], e[2][k1]};
            Bfly<3>::run(t);
            v[k1] = t[0]; v[k1 + 4] = t[1]; v[k1 + 8] = t[2];
        }
    }
};

// One Stockham pass of radix R over `nlines` lines of length N, butterflies tid, tid+nthreads, ...
//   ns = product of the radices of the earlier passes (1 for the first pass).
//   ld(line, idx) -> cd      reads element idx of the line in the pass's input
//   st(line, idx, value)     writes element idx of the line in the pass's output (idx is the final frequency
//                            index when this is the last pass)
//   tw[t] = exp(-2 pi i t/N), t = 0..N-1
//   LINE_FAST = false: consecutive threads take consecutive butterflies of one line (coalesced along the line);
//   LINE_FAST = true : consecutive threads take the same butterfly of consecutive lines (for data stored
//                      [element][line], every access is then contiguous and the twiddles are warp-uniform).
//   NC, NSC > 0 fix N and ns at compile time (the runtime arguments are then ignored).
template <int R, bool LINE_FAST, int NC = 0, int NSC = 0, class LD, class ST>
HD void fft_pass(int tid, int nthreads, int nlines, int N_rt, int ns_rt, const cd *tw, LD ld, ST st) {
    const int N = NC > 0 ? NC : N_rt;
    const int ns = NSC > 0 ? NSC : ns_rt;
    const int nb = N / R;            // butterflies per line
    const int total = nlines * nb;
    const int tstep = nb / ns;       // N / (ns R)
    for (int idx = tid; idx < total; idx += nthreads) {
        int line, j;
        if (LINE_FAST) {
            j = idx / nlines;
            line = idx - j * nlines;
        } else {
            line = idx / nb;
            j = idx - line * nb;
        }
        cd v[R];
#pragma unroll
        for (int s = 0; s < R; s++) v[s] = ld(line, j + s * nb);
        const int k = j % ns;
        if (ns > 1) {
            const int t1 = k * tstep;
#pragma unroll
            for (int s = 1; s < R; s++) v[s] = h_mul(v[s], tw[s * t1]);
        }
        Bfly<R>::run(v);
        const int j0 = (j - k) * R + k;
#pragma unroll
        for (int s = 0; s < R; s++) st(line, j0 + s * ns, v[s]);
    }
}

template <bool LINE_FAST, class LD, class ST>
HD void fft_pass_r(int R, int tid, int nthreads, int nlines, int N, int ns, const cd *tw, LD ld, ST st) {
    switch (R) {
        case 2: fft_pass<2, LINE_FAST, 0, 0>(tid, nthreads, nlines, N, ns, tw, ld, st); break;
        case 3: fft_pass<3, LINE_FAST, 0, 0>(tid, nthreads, nlines, N, ns, tw, ld, st); break;
        case 4: fft_pass<4, LINE_FAST, 0, 0>(tid, nthreads, nlines, N, ns, tw, ld, st); break;
        case 5: fft_pass<5, LINE_FAST, 0, 0>(tid, nthreads, nlines, N, ns, tw, ld, st); break;
        case 6: fft_pass<6, LINE_FAST, 0, 0>(tid, nthreads, nlines, N, ns, tw, ld, st); break;
        case 7: fft_pass<7, LINE_FAST, 0, 0>(tid, nthreads, nlines, N, ns, tw, ld, st); break;
        default: fft_pass<8, LINE_FAST, 0, 0>(tid, nthreads, nlines, N, ns, tw, ld, st); break;
    }
}

// Radix plan for a length with prime factors 2,3,5,7 only; ok = false otherwise.  Prefers few, large passes.
// constexpr so that the kernels specialised on a grid length get their radices at compile time.
struct FftPlanResult {
    FftPlan plan;
    bool ok;
};

__host__ __device__ constexpr FftPlanResult fft_plan_c(int n) {
    FftPlanResult out{};
    out.plan.n = n;
    out.plan.npass = 0;
    out.ok = false;
    if (n < 1) return out;
    int m = n;
    int c2 = 0, c3 = 0, c5 = 0, c7 = 0;
    while (m % 2 == 0) { m /= 2; c2++; }
    while (m % 3 == 0) { m /= 3; c3++; }
    while (m % 5 == 0) { m /= 5; c5++; }
    while (m % 7 == 0) { m /= 7; c7++; }
    if (m != 1) return out;
    int r[32] = {};
    int nr = 0;
    while (c2 >= 3) { r[nr++] = 8; c2 -= 3; }
    if (c2 == 2) { r[nr++] = 4; c2 = 0; }
    if (c2 == 1 && c3 >= 1) { r[nr++] = 6; c2 = 0; c3--; }
    while (c7 > 0) { r[nr++] = 7; c7--; }
    while (c5 > 0) { r[nr++] = 5; c5--; }
    while (c3 > 0) { r[nr++] = 3; c3--; }
    if (c2 == 1) r[nr++] = 2;
    // n == 1: npass = 0, callers treat the axis as a copy
    if (nr > FFT_MAX_PASSES) return out;
    out.plan.npass = nr;
    for (int i = 0; i < nr; i++) out.plan.radix[i] = r[i];
    out.ok = true;
    return out;
}

static inline bool fft_make_plan(int n, FftPlan *p) {
    const FftPlanResult r = fft_plan_c(n);
    *p = r.plan;
    return r.ok;
}
