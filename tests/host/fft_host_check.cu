// Host-side check of the register butterflies and Stockham passes of csrc/fft.cuh against a direct DFT
// (long double).  Built by tests/test_fft_host.py with nvcc, runs on the CPU (no GPU needed).
#include <math.h>
#include <stdio.h>
#include <vector>

#include "../../paper_1307_8052_b200/csrc/fft.cuh"

static double check_bfly(int R, void (*run)(cd *)) {
    std::vector<cd> v(R), ref(R);
    for (int i = 0; i < R; i++) v[i] = make_double2(sin(1.0 + 3.7 * i), cos(0.3 + 1.9 * i * i));
    for (int k = 0; k < R; k++) {
        long double re = 0, im = 0;
        for (int j = 0; j < R; j++) {
            const long double a = -2.0L * 3.14159265358979323846264338327950288L * (long double)((j * k) % R) / R;
            re += v[j].x * cosl(a) - v[j].y * sinl(a);
            im += v[j].x * sinl(a) + v[j].y * cosl(a);
        }
        ref[k] = make_double2((double)re, (double)im);
    }
    run(v.data());
    double err = 0;
    for (int k = 0; k < R; k++) err = fmax(err, hypot(v[k].x - ref[k].x, v[k].y - ref[k].y));
    return err;
}

// full mixed-radix line through fft_pass (ping-pong buffers), natural-order output
static double check_line(int n) {
    FftPlan p;
    if (!fft_make_plan(n, &p)) return -1.0;
    std::vector<cd> a(n), b(n), tw(n), x(n);
    for (int i = 0; i < n; i++) {
        x[i] = a[i] = make_double2(sin(0.7 * i + 0.1), cos(1.3 * i));
        const long double ang = -2.0L * 3.14159265358979323846264338327950288L * i / n;
        tw[i] = make_double2((double)cosl(ang), (double)sinl(ang));
    }
    int ns = 1;
    cd *src = a.data(), *dst = b.data();
    for (int ps = 0; ps < p.npass; ps++) {
        auto ld = [&](int, int i) { return src[i]; };
        auto st = [&](int, int i, cd v) { dst[i] = v; };
        fft_pass_r<false>(p.radix[ps], 0, 1, 1, n, ns, tw.data(), ld, st);
        ns *= p.radix[ps];
        cd *t = src; src = dst; dst = t;
    }
    double err = 0;
    for (int k = 0; k < n; k++) {
        long double re = 0, im = 0;
        for (int j = 0; j < n; j++) {
            const long double ang = -2.0L * 3.14159265358979323846264338327950288L * (long double)(((long)j * k) % n) / n;
            re += x[j].x * cosl(ang) - x[j].y * sinl(ang);
            im += x[j].x * sinl(ang) + x[j].y * cosl(ang);
        }
        err = fmax(err, hypot(src[k].x - (double)re, src[k].y - (double)im));
    }
    return err;
}

int main() {
    printf("bfly 2 %.3e\n", check_bfly(2, Bfly<2>::run));
    printf("bfly 3 %.3e\n", check_bfly(3, Bfly<3>::run));
    printf("bfly 4 %.3e\n", check_bfly(4, Bfly<4>::run));
    printf("bfly 5 %.3e\n", check_bfly(5, Bfly<5>::run));
    printf("bfly 6 %.3e\n", check_bfly(6, Bfly<6>::run));
    printf("bfly 7 %.3e\n", check_bfly(7, Bfly<7>::run));
    printf("bfly 8 %.3e\n", check_bfly(8, Bfly<8>::run));
    printf("bfly 12 %.3e\n", check_bfly(12, Bfly<12>::run));
    const int lens[] = {1, 2, 16, 24, 40, 48, 56, 60, 64, 168, 192, 210, 45};
    for (int n : lens) printf("line %d %.3e\n", n, check_line(n));
    return 0;
}
