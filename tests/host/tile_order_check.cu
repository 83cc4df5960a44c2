// Host-side check of the work-item order of rank_k3m_kernel (csrc/rank_k3m.cuh): rk3_tile_order(ng) must be a permutation
// of the lower-triangle tiles, never increasing in work, and rk3_tile_units(ti, tj, ng) must count exactly the 8-row x
// 16-column warp blocks of a tile that hold an element of the lower triangle of an ng x ng matrix -- against a plain walk
// over the elements.  Built by tests/test_fft_host.py with nvcc, runs on the CPU.  Prints "<sizes> <bad>".
#include <stdio.h>
#include <vector>

#include "../../paper_1307_8052_b200/csrc/rank_k3m.cuh"

static long check(int ng) {
    using namespace rk3;
    long bad = 0;
    const int nt = (ng + T - 1) / T;
    const std::vector<int32_t> order = rk3_tile_order(ng);
    bad += (int)order.size() != nt * (nt + 1) / 2;
    std::vector<int> seen(order.size(), 0), work(order.size(), 0);
    for (int ti = 0; ti < nt; ti++)
        for (int tj = 0; tj <= ti; tj++) {
            // the definition: blocks (8 rows x 16 columns, as the warps are laid out) with an element g >= g' < ng inside.
            // The kernel may compute a few more (a warp skips whole 8-row blocks, not single 16-column halves), never fewer.
            int need = 0;
            for (int rb = 0; rb < T / 8; rb++)
                for (int cb = 0; cb < T / 16; cb++) {
                    bool any = false;
                    for (int r = ti * T + rb * 8; r < ti * T + rb * 8 + 8 && !any; r++)
                        for (int c = tj * T + cb * 16; c < tj * T + cb * 16 + 16; c++)
                            if (r < ng && c < ng && c <= r) { any = true; break; }
                    need += any;
                }
            const int got = rk3_tile_units(ti, tj, ng);
            bad += got < need || got > T / 8 * (T / 16);
            if (ti != tj && ti * T + T <= ng) bad += got != 32;   // a full tile off the diagonal: all 32 blocks
            work[ti * (ti + 1) / 2 + tj] = got;
        }
    for (size_t i = 0; i < order.size(); i++) {
        if (order[i] < 0 || order[i] >= (int32_t)order.size()) { bad++; continue; }
        seen[order[i]]++;
        if (i > 0 && work[order[i]] > work[order[i - 1]]) bad++;
    }
    for (int v : seen) bad += v != 1;
    return bad;
}

int main() {
    long bad = 0;
    int n = 0;
    for (int ng = 1; ng <= 700; ng++, n++) bad += check(ng);
    const int more[] = {1200, 3004, 5001, 4096, 4097};
    for (int ng : more) { bad += check(ng); n++; }
    printf("%d %ld\n", n, bad);
    return bad != 0;
}
