// Host-side check of the work-item map of pd_zy_kernel (csrc/pair_density_zy.cuh): pdzy_plan_units + pdzy_unit must
// enumerate, for every launch [p_begin, p_begin + p_count) of a batch whose rows are mlen pairs long, exactly the groups of
// <= G consecutive pairs that never cross a row boundary, in order -- the closed form with magic-number divisions against a
// plain walk over the pairs.  Also pdzy_fastdiv against the integer division.  Built by tests/test_fft_host.py with nvcc,
// runs on the CPU.
#include <stdio.h>
#include <stdlib.h>
#include <algorithm>

#include "../../paper_1307_8052_b200/csrc/pair_density_zy.cuh"

template <int G>
static long check(int p_begin, int p_count, int mlen, int N1) {
    PdZyParams P;
    P.p_begin = p_begin; P.p_count = p_count; P.mlen = mlen; P.N1 = N1;
    pdzy_plan_units(P, G);
    long bad = 0;
    int u = 0, p = p_begin;
    const int p_end = p_begin + p_count;
    while (p < p_end) {   // the definition: walk the pairs, cut at row ends and every G pairs
        const int row = p / mlen, rend = std::min((row + 1) * mlen, p_end), cnt = std::min(G, rend - p);
        int gp, gc, gr;
        pdzy_unit<G>(P, u, gp, gc, gr);
        bad += (gp != p) + (gc != cnt) + (gr != row);
        p += cnt;
        u++;
    }
    bad += (u != P.n_units);
    // items w = u N1 + j1 are split with the same division
    for (int w = 0; w < P.n_units * N1; w += 1 + (w % 7)) bad += (pdzy_fastdiv(w, P.magic_n1) != w / N1);
    return bad;
}

int main() {
    long bad = 0, cases = 0;
    srand(12345);
    for (int it = 0; it < 20000; it++) {
        const int mlen = 1 + rand() % 700, rows = 1 + rand() % 17, K = mlen * rows;
        const int p_begin = rand() % K, p_count = 1 + rand() % (K - p_begin), N1 = 1 + rand() % 200;
        bad += check<1>(p_begin, p_count, mlen, N1) + check<2>(p_begin, p_count, mlen, N1) + check<4>(p_begin, p_count, mlen, N1);
        cases += 3;
    }
    // the shapes of BASELINE.json configs[4] with its 4 GB scratch split: 8 x 1024 pairs, second launch starts mid-row
    bad += check<2>(7050, 1142, 1024, 48) + check<2>(0, 7050, 1024, 48) + check<4>(0, 2400, 300, 24) + check<4>(0, 7200, 600, 56);
    for (long long d = 1; d < 5000; d++)
        for (long long x : {0ll, 1ll, d - 1, d, d + 1, 2 * d - 1, 1000003ll, 2147483647ll})
            bad += (pdzy_fastdiv((int)x, pdzy_magic((int)d)) != (int)(x / d));
    printf("%ld %ld\n", cases, bad);
    return bad != 0;
}
