// librpa_chi0.so -- host orchestration and C ABI of the chi0 / RPA hot path (include/rpa_chi0.h).
// Everything on the path runs in the kernels of pair_density.cuh, paw.cuh, rank_k.cuh and energy.cuh; this file
// builds the sphere tables, carves the caller's workspace, plans the batches and enqueues the launches.
#include <cuda.h>
#include <cuda_runtime.h>
#include <limits.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/rpa_chi0.h"
#include "common.cuh"
#include "energy.cuh"
#include "fft.cuh"
#include "pair_density.cuh"
#include "pair_density_zy.cuh"
#include "orbitals.cuh"
#include "optical.cuh"
#include "paw.cuh"
#include "rank_k.cuh"
#include "rank_k3m.cuh"
#include "rank_k_i8.cuh"

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(expr)                                                                                      \
    do {                                                                                                    \
        cudaError_t e_ = (expr);                                                                            \
        if (e_ != cudaSuccess) return fail(RPA_ERR_CUDA, "%s: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

constexpr int DEFAULT_BATCH = 8192;
constexpr int MAX_SLOTS = 16;          // occupied bands per batch
constexpr int I8_MIN_NG = 768, I8_MIN_K = 1024;  // below: the FP64 tensor kernel is faster (measured: nG = 401, K = 2400 loses)
constexpr int MAX_BANDS = 1 << 17;     // eps/f scratch
constexpr int MAX_ATOMS = 4096;
constexpr int MAX_PROJ = 1 << 16;
constexpr int EC_DEFAULT_LANES = 2;
constexpr int EC_MAX_LANES = 4;       // concurrent shares of a group in rpa_ec_q
constexpr int EC_GROUP = 16;           // frequencies factorised together in rpa_ec_q
constexpr size_t I_BUDGET = (size_t)4 << 30; // pruned intermediate of a whole batch when it fits (fewer, larger launches beat L2 residency)
constexpr int NSTAGE = 6;
constexpr int K_ALIGN = 32;            // pairs per batch are padded to the chunk size of both rank-K kernels (16, 32)
static_assert(K_ALIGN % rk::KC == 0 && K_ALIGN % rk3::KC == 0, "batch padding");

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Sphere {
    int ng = 0;
    std::vector<int32_t> g;    // [ng][3]
    std::vector<double> K2;    // |q+G|^2
    std::vector<double> Kc;    // [ng][3] Cartesian q+G
    int gmin[3] = {0, 0, 0}, gmax[3] = {0, 0, 0};
    // the (g2, g3) columns of the bounding box that hold at least one sphere point, ascending in g2i ng3 + g3i: the pruned
    // transforms keep only these after the y axis (configs[2]: 73 of 121, configs[1]: 147 of 195)
    std::vector<int32_t> coltab;   // (g2i << 16) | g3i
    std::vector<int32_t> rowtab;   // [ng2 + 1]: first column of every g2i
    int ncols = 0;
};

void recip_lattice(const double A[9], double B[9], double *vol) {
    // B = 2 pi A^-T: rows b_i = 2 pi (a_j x a_k) / det
    const double *a1 = A, *a2 = A + 3, *a3 = A + 6;
    double c23[3] = {a2[1] * a3[2] - a2[2] * a3[1], a2[2] * a3[0] - a2[0] * a3[2], a2[0] * a3[1] - a2[1] * a3[0]};
    double c31[3] = {a3[1] * a1[2] - a3[2] * a1[1], a3[2] * a1[0] - a3[0] * a1[2], a3[0] * a1[1] - a3[1] * a1[0]};
    double c12[3] = {a1[1] * a2[2] - a1[2] * a2[1], a1[2] * a2[0] - a1[0] * a2[2], a1[0] * a2[1] - a1[1] * a2[0]};
    const double det = a1[0] * c23[0] + a1[1] * c23[1] + a1[2] * c23[2];
    const double s = 2.0 * M_PI / det;
    for (int i = 0; i < 3; i++) {
        B[i] = s * c23[i];
        B[3 + i] = s * c31[i];
        B[6 + i] = s * c12[i];
    }
    *vol = fabs(det);
}

// Sphere of Table 1 step 6: strict |g_i| < N_i/2, |q+G|^2/2 <= ecut, ascending flat FFT index.
void build_sphere(const int32_t grid[3], const double B[9], const double q[3], double ecut, Sphere *sp) {
    sp->ng = 0;
    sp->g.clear(); sp->K2.clear(); sp->Kc.clear();
    bool first = true;
    for (int i1 = 0; i1 < grid[0]; i1++) {
        const int g1 = (2 * i1 < grid[0]) ? i1 : i1 - grid[0];
        if (2 * abs(g1) >= grid[0]) continue;
        for (int i2 = 0; i2 < grid[1]; i2++) {
            const int g2 = (2 * i2 < grid[1]) ? i2 : i2 - grid[1];
            if (2 * abs(g2) >= grid[1]) continue;
            for (int i3 = 0; i3 < grid[2]; i3++) {
                const int g3 = (2 * i3 < grid[2]) ? i3 : i3 - grid[2];
                if (2 * abs(g3) >= grid[2]) continue;
                const double x = q[0] + g1, y = q[1] + g2, z = q[2] + g3;
                const double K[3] = {x * B[0] + y * B[3] + z * B[6], x * B[1] + y * B[4] + z * B[7],
                                     x * B[2] + y * B[5] + z * B[8]};
                const double K2 = K[0] * K[0] + K[1] * K[1] + K[2] * K[2];
                if (0.5 * K2 <= ecut) {
                    const int gv[3] = {g1, g2, g3};
                    for (int d = 0; d < 3; d++) {
                        sp->g.push_back(gv[d]);
                        sp->Kc.push_back(K[d]);
                        if (first || gv[d] < sp->gmin[d]) sp->gmin[d] = gv[d];
                        if (first || gv[d] > sp->gmax[d]) sp->gmax[d] = gv[d];
                    }
                    first = false;
                    sp->K2.push_back(K2);
                    sp->ng++;
                }
            }
        }
    }
    if (sp->ng > 0) {
        const int ng2 = sp->gmax[1] - sp->gmin[1] + 1, ng3 = sp->gmax[2] - sp->gmin[2] + 1;
        std::vector<char> used((size_t)ng2 * ng3, 0);
        for (int s = 0; s < sp->ng; s++) used[(size_t)(sp->g[3 * s + 1] - sp->gmin[1]) * ng3 + (sp->g[3 * s + 2] - sp->gmin[2])] = 1;
        sp->coltab.clear();
        sp->rowtab.assign(ng2 + 1, 0);
        for (int o = 0; o < ng2; o++) {
            sp->rowtab[o] = (int32_t)sp->coltab.size();
            for (int c = 0; c < ng3; c++)
                if (used[(size_t)o * ng3 + c]) sp->coltab.push_back((o << 16) | c);
        }
        sp->rowtab[ng2] = (int32_t)sp->coltab.size();
        sp->ncols = (int)sp->coltab.size();
    }
}

struct Layout {
    size_t S, Nbuf, NS, w, I, T, M, Lt, wneg, tw1, tw2, tw3, box2s, coltab, rowtab, Kc, omega, wt, band, R, aj_atom, aj_j, atom_poff, atom_ni,
        atom_qoff, v, e, tr, logdet, flag, ec, pwtab, rkorder, total;
    int64_t ldS, ldn, ldw;
    int Kmax, sub_pairs, ec_group;
    size_t I_pair_bytes;
};

bool valid_dims(const int32_t grid[3], const double cell[9], const double q[3], double ecut, int n_omega) {
    if (!grid || !cell || !q) return false;
    if (grid[0] < 1 || grid[1] < 1 || grid[2] < 1) return false;
    if ((int64_t)grid[0] * grid[1] * grid[2] > (int64_t)1 << 30) return false;
    if (!(ecut > 0.0) || n_omega < 1) return false;
    return true;
}

void make_layout(const int32_t grid[3], const Sphere &sp, int n_omega, int max_batch, int max_proj, Layout *L) {
    const int ng = sp.ng;
    int Kmax = max_batch <= 0 ? DEFAULT_BATCH : max_batch;
    Kmax = (int)align_up((size_t)std::max(Kmax, K_ALIGN), K_ALIGN);
    L->Kmax = Kmax;
    L->ldS = ng;
    L->ldn = (int64_t)align_up((size_t)ng, 8);
    L->ldw = Kmax;
    const int nb2 = (sp.gmax[1] - sp.gmin[1] + 1) * (sp.gmax[2] - sp.gmin[2] + 1);
    const int ng1 = sp.gmax[0] - sp.gmin[0] + 1;
    L->I_pair_bytes = (size_t)grid[0] * nb2 * sizeof(cd);
    L->sub_pairs = (int)std::max<size_t>(1, std::min<size_t>((size_t)Kmax, I_BUDGET / std::max<size_t>(1, L->I_pair_bytes)));
    L->ec_group = std::min(EC_GROUP, n_omega);
    size_t off = 0;
    auto take = [&](size_t bytes) {
        size_t o = off;
        off = align_up(off + bytes, 256);
        return o;
    };
    L->S = take((size_t)n_omega * ng * L->ldS * sizeof(cd));
    L->Nbuf = take((size_t)Kmax * L->ldn * sizeof(cd));
    L->NS = take((size_t)Kmax * L->ldn * sizeof(double));   // Re + Im of N: third operand plane of rank_k3m_kernel
    L->w = take((size_t)n_omega * L->ldw * sizeof(double));
    L->I = take((size_t)L->sub_pairs * L->I_pair_bytes);
    L->T = take((size_t)MAX_SLOTS * std::max(max_proj, 0) * L->ldn * sizeof(cd));
    L->M = take((size_t)L->ec_group * ng * ng * sizeof(cd));
    L->Lt = take(2 * (size_t)L->ec_group * CH_P * CH_NB * L->ldn * sizeof(cd));   // two blocks of CH_P panels (look-ahead)
    L->wneg = take((size_t)L->ec_group * CH_P * CH_NB * sizeof(double));
    L->tw1 = take((size_t)grid[0] * sizeof(cd));
    L->tw2 = take((size_t)grid[1] * sizeof(cd));
    L->tw3 = take((size_t)grid[2] * sizeof(cd));
    L->box2s = take((size_t)ng1 * nb2 * sizeof(int32_t));
    L->coltab = take((size_t)nb2 * sizeof(int32_t));
    L->rowtab = take((size_t)(sp.gmax[1] - sp.gmin[1] + 2) * sizeof(int32_t));
    L->Kc = take((size_t)ng * 3 * sizeof(double));
    L->omega = take((size_t)n_omega * sizeof(double));
    L->wt = take((size_t)n_omega * sizeof(double));
    L->band = take((size_t)MAX_BANDS * 2 * sizeof(double));
    L->R = take((size_t)MAX_ATOMS * 3 * sizeof(double));
    L->aj_atom = take((size_t)std::max(max_proj, 1) * sizeof(int32_t));
    L->aj_j = take((size_t)std::max(max_proj, 1) * sizeof(int32_t));
    L->atom_poff = take((size_t)MAX_ATOMS * sizeof(int32_t));
    L->atom_ni = take((size_t)MAX_ATOMS * sizeof(int32_t));
    L->atom_qoff = take((size_t)MAX_ATOMS * sizeof(int64_t));
    L->v = take((size_t)ng * sizeof(double));
    L->e = take((size_t)n_omega * sizeof(double));
    L->tr = take((size_t)EC_GROUP * sizeof(double));
    L->logdet = take((size_t)EC_GROUP * sizeof(double));
    L->flag = take((size_t)EC_GROUP * sizeof(int));
    L->ec = take(sizeof(double));
    L->pwtab = take((size_t)grid[0] * grid[1] * grid[2] * sizeof(int32_t));   // plane-wave box -> coefficient index (rpa_pw_to_grid), kept between calls
    L->rkorder = take((size_t)((ng + rk3::T - 1) / rk3::T) * ((ng + rk3::T - 1) / rk3::T + 1) / 2 * sizeof(int32_t));   // rank_k3m_kernel: tiles, heaviest first
    L->total = off;
}

struct StageEvent {
    int stage;
    cudaEvent_t a, b;
};

}  // namespace

// One call's arguments (rpa_chi0_add_kpoint, rpa_chi0_add_kpoint_optical when grad != NULL, or the streamed variant)
struct AddArgs {
    double kweight;
    int32_t n_occ;
    const void *psi_occ;
    int32_t n_unocc;
    const void *psi_unocc;
    const double *eps_occ, *eps_unocc, *f_occ, *f_unocc;
    int32_t n_atoms;
    const int32_t *n_proj;
    const void *P_occ, *P_unocc, *Q;
    const double *R_cart, *qdir;
    const void *grad;
};

struct rpa_chi0 {
    cudaStream_t stream = nullptr;
    int32_t grid[3];
    double cell[9], B[9], q[3], vol, ecut;
    int n_omega;                       // accumulator slots: the frequencies, or 2 per frequency on the real axis
    int n_freq;                        // frequencies the caller sees
    double eta = -1.0;                 // > 0: real-axis handle, chi0 at omega + i eta (slot 2i: Re w, slot 2i+1: Im w)
    bool has_wt;
    std::vector<double> omega, wt;
    Sphere sp;
    Layout L;
    int max_proj;
    FftPlan pz, py;
    int RC, pd_threads, pd_nbuf;
    PdPlaneKernel pd_kernel = nullptr;
    size_t pd_smem;
    PdZyKernel zy_kernel = nullptr;   // low-instruction-count z+y kernel (planes that fit one CTA), else pd_kernel
    int zy_G = 1, zy_threads = 0, zy_ctas_per_sm = 1, n_sm = 148;
    double spin_deg = 2.0;             // prefactor s of chi0 = (s/Omega) S: 2 spin-paired (A3), 1 per explicit spin channel
    bool q0 = false;                   // q = 0: pair densities need the optical-limit head (rpa_chi0_add_kpoint_optical)
    int idx0 = -1;                     // sphere index of G = 0 when q0
    // rank-K kernel of the chi0 accumulation (rpa_chi0_set_rank_k_mode; default: FP64 tensor cores, 3-multiplication)
    bool use_i8 = false;               // RPA_RANK_K_I8: int8-sliced rank-K on tcgen05 (rank_k_i8.cuh) for large batches
    int i8_digits = 7;
    bool i8_cluster = true;            // clusters of 2 CTAs multicast the row-block digits (RPA_RANK_K_FLAG_NO_CLUSTER: off)
    bool i8_force = false;             // RPA_RANK_K_FLAG_ALL_BATCHES: also for batches below I8_MIN_NG / I8_MIN_K
    bool i8_attr_set = false;          // cudaFuncSetAttribute done for the rank_k_i8_kernel instances
    std::vector<int2> i8_tiles;        // (row block, column block) tiles that meet the lower triangle
    CUtensorMap nmap, smap;            // 2-D FP64 tensor maps for rank_k3m_kernel over N (dims (2 ldn, Kmax), box (132, 16)) and NS ((ldn, Kmax), (68, 16))
    bool use_3m = true;                // rank_k3m_kernel (3-multiplication complex product); false: rank_k_kernel<true> (4M)
    int64_t i8_batches = 0, fp64_batches = 0;   // batches each rank-K path has taken (rpa_chi0_rank_k_batches)
    int ec_lanes = EC_DEFAULT_LANES;   // rpa_chi0_set_ec_lanes
    struct EcGraph { int nm, lanes; cudaGraphExec_t exec; int64_t launches; };
    std::vector<EcGraph> ec_graphs;    // captured factorisations of rpa_ec_q, one per (matrices in the group, lanes)
    bool ec_use_graph = true;
    bool ec_tile32 = true;             // chain updates of rpa_ec_q by chol_update32_kernel (RPA_EC_FLAG_WIDE_TILES: rank_k_kernel<false>)
    cudaStream_t side = nullptr;       // panel factorisations of rpa_ec_q run here, ahead of the trailing updates
    cudaEvent_t ev_panel[2] = {nullptr, nullptr}, ev_col = nullptr, ev_fork = nullptr;
    // further lanes of rpa_ec_q (each factorises its share of the matrices of a group on its own stream pair)
    cudaStream_t xmain[EC_MAX_LANES - 1] = {}, xside[EC_MAX_LANES - 1] = {};
    cudaEvent_t xev_panel[EC_MAX_LANES - 1][2] = {}, xev_col[EC_MAX_LANES - 1] = {}, xev_join[EC_MAX_LANES - 1] = {};
    size_t zy_smem = 0;
    // rpa_pw_to_grid: the index table of the last g_pw, kept on the device (L.pwtab) while the caller passes the same vectors
    std::vector<int32_t> pw_g, pw_table;
    int pw_qmin[3] = {0, 0, 0};
    int64_t pw_nq[3] = {0, 0, 0};
    // streamed k-point (rpa_chi0_add_kpoint_begin / _pairs / _end): the open call's arguments (the host arrays among them are
    // not used after _begin), its projector count and the first unoccupied band not yet given to _pairs
    bool pend_open = false;
    AddArgs pend = {};
    int pend_ptot = 0, pend_m_next = 0;
    unsigned char *ws;
    // profiling
    bool prof = false;
    std::vector<StageEvent> events;
    std::vector<cudaEvent_t> pool;
    double stage_ms[NSTAGE] = {0, 0, 0, 0, 0, 0};
    int64_t stage_launches[NSTAGE] = {0, 0, 0, 0, 0, 0};
    int64_t launches = 0;  // every kernel launch enqueued through this handle

    template <class T>
    T *ptr(size_t off) const { return reinterpret_cast<T *>(ws + off); }
};

namespace {

cudaEvent_t get_event(rpa_chi0 *h) {
    if (!h->pool.empty()) {
        cudaEvent_t e = h->pool.back();
        h->pool.pop_back();
        return e;
    }
    cudaEvent_t e;
    cudaEventCreate(&e);
    return e;
}

struct StageTimer {
    rpa_chi0 *h;
    int stage;
    cudaEvent_t a = nullptr, b = nullptr;
    StageTimer(rpa_chi0 *h_, int stage_, int launches) : h(h_), stage(stage_) {
        h->stage_launches[stage] += h->prof ? launches : 0;
        h->launches += launches;
        if (h->prof) {
            a = get_event(h);
            b = get_event(h);
            cudaEventRecord(a, h->stream);
        }
    }
    ~StageTimer() {
        if (h->prof) {
            cudaEventRecord(b, h->stream);
            h->events.push_back({stage, a, b});
        }
    }
};

int drain_events(rpa_chi0 *h) {
    for (auto &ev : h->events) {
        CUDA_TRY(cudaEventSynchronize(ev.b));
        float ms = 0.f;
        CUDA_TRY(cudaEventElapsedTime(&ms, ev.a, ev.b));
        h->stage_ms[ev.stage] += ms;
        h->pool.push_back(ev.a);
        h->pool.push_back(ev.b);
    }
    h->events.clear();
    return RPA_OK;
}

int ntiles_lower(int n, int t) {
    const int nt = (n + t - 1) / t;
    return nt * (nt + 1) / 2;
}

// K slices of the rank-K launch: one CTA per SM, `units` equal work items (tile x frequency pair).  With s slices
// the grid needs ceil(units s / n_sm) rounds of 1/s of an item each; take the s that minimises that time, charging
// 3 % per extra slice for its prologue / atomic epilogue (measured on the 448 items of configs[2], K = 2400: 2 / 3 / 4
// slices 0.787 / 0.781 / 0.807 ms, one 0.869), and keep at least min_chunks chunks (512 pairs) per slice.
int pick_ksplit(int units, int nchunks, int n_sm, double *cost_out = nullptr, int min_chunks = 16) {
    int best = 1;
    double best_cost = 1e300;
    for (int s = 1; s <= 8 && nchunks / s >= min_chunks; s++) {
        const double rounds = (double)(((int64_t)units * s + n_sm - 1) / n_sm) / s;
        const double cost = rounds * (1.0 + 0.03 * (s - 1));
        if (cost < best_cost * (1.0 - 1e-9)) { best_cost = cost; best = s; }
    }
    if (cost_out) *cost_out = best_cost;   // in units of one full-K item
    return best;
}

// rank_k_i8_kernel<S, 2> as clusters of two CTAs along x (tiles come in pairs of one row block), or <S, 1> plain
template <int S>
cudaError_t launch_i8(bool cluster, dim3 grid, cudaStream_t st, const int8_t *PL, const int8_t *PR, int nkb, int ncb,
                      const int2 *tiles, const double *invL, const double *invR, int ng, int ngp, cd *Sacc, int64_t ldS,
                      int64_t strideS) {
    if (!cluster) {
        rank_k_i8_kernel<S, 1><<<grid, rki8::THREADS, rki8::smem_bytes(S), st>>>(PL, PR, nkb, ncb, tiles, invL, invR, ng, ngp, Sacc, ldS, strideS);
        return cudaGetLastError();
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = dim3(rki8::THREADS);
    cfg.dynamicSmemBytes = rki8::smem_bytes(S);
    cfg.stream = st;
    cudaLaunchAttribute attr;
    attr.id = cudaLaunchAttributeClusterDimension;
    attr.val.clusterDim.x = 2;
    attr.val.clusterDim.y = 1;
    attr.val.clusterDim.z = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, rank_k_i8_kernel<S, 2>, PL, PR, nkb, ncb, tiles, invL, invR, ng, ngp, Sacc, ldS, strideS);
}

// Launch plan of the plane kernel: rows per chunk, threads, dynamic shared memory.
//  run-time radix passes with cp.async staging, two CTAs per SM preferred (the specialised pd_zy_kernel, when one
//  exists for the plane shape, is planned by plan_zy_kernel).
// Returns false if even one z line per chunk does not fit.
template <class C, class K>
void try_zy(rpa_chi0 *h, K kernel, int G, int minb) {
    const int ng2 = h->sp.gmax[1] - h->sp.gmin[1] + 1, ng3 = h->sp.gmax[2] - h->sp.gmin[2] + 1;
    if (!C::box_ok(h->sp.gmin[2], ng3)) return;
    const size_t smem = C::smem_bytes(ng2, ng3);
    if (smem > 200 * 1024) return;
    h->zy_kernel = kernel;
    h->zy_G = G;
    h->zy_threads = C::NTH;
    h->zy_smem = smem;
    h->zy_ctas_per_sm = (int)std::max<size_t>(1, std::min<size_t>((size_t)minb, (227 * 1024) / (smem + 1024)));
}

// Specialisations of the z+y kernel for the plane shapes of BASELINE.json configs[0..2] (G pairs per unit and CTAs
// per SM tuned on B200: 8 warps per SM without spills beat 12 with); other shapes take the pd_plane kernels.
void plan_zy_kernel(rpa_chi0 *h) {
    const int N2 = h->grid[1], N3 = h->grid[2];
    h->zy_kernel = nullptr;
#define ZY(N3_, NA3_, DLO_, DHI_, N2_, NA2_, NW_, LPW_, G_, MINB_, ...)                \
    try_zy<PdZy<N3_, NA3_, DLO_, DHI_, N2_, NA2_, NW_, LPW_, G_>>(                     \
        h, pd_zy_kernel<N3_, NA3_, DLO_, DHI_, N2_, NA2_, NW_, LPW_, G_, MINB_, ##__VA_ARGS__>, G_, MINB_)
    if (N2 == 60 && N3 == 64) ZY(64, 8, -1, 0, 60, 12, 4, 4, 4, 2, true);
    // 24-point lines as 6 x 4 (4 lanes per line, 8 lines per warp: every lane busy, 64 contiguous bytes per line and load
    // instruction) and 12 x 2 in y: 1.58 -> 1.33 ms per 8 k-points of configs[2] against the 8 x 3 / 8 x 3 split
    else if (N2 == 24 && N3 == 24) ZY(24, 6, -1, 0, 24, 12, 3, 8, 4, 3);
    else if (N2 == 16 && N3 == 16) ZY(16, 8, -1, 0, 16, 8, 1, 16, 4, 8);
    else if (N2 == 40 && N3 == 168) ZY(168, 12, -2, 1, 40, 8, 4, 2, 1, 2);
    else if (N2 == 48 && N3 == 192) ZY(192, 12, -3, 2, 48, 12, 8, 2, 2, 1, true);
#undef ZY
}

bool plan_plane_kernel(rpa_chi0 *h) {
    const int N2 = h->grid[1], N3 = h->grid[2];
    const int ng3 = h->sp.gmax[2] - h->sp.gmin[2] + 1;
    plan_zy_kernel(h);
    const int N3p = N3 + (N3 >> 3) + 1;
    const int nbuf = h->pz.npass >= 3 ? 2 : (h->pz.npass == 2 ? 1 : 0);
    h->pd_nbuf = nbuf;
    h->pd_kernel = pd_plane_kernel<0, 0>;   // run-time radix passes: any 2-3-5-7 plane shape
    const size_t ysz = (size_t)ng3 * N2;
    const size_t fixed = ((size_t)N3 + N2 + 2 * ysz) * sizeof(cd);
    const size_t per_row = (4 * (size_t)N3 + (size_t)nbuf * N3p) * sizeof(cd);
    const size_t caps[3] = {72 * 1024, 110 * 1024, 224 * 1024};   // 3, 2, 1 CTAs per SM
    int rc = 0;
    for (int t = 1; t < 3 && rc == 0; t++) {
        if (caps[t] <= fixed + per_row) continue;
        const int r = (int)((caps[t] - fixed) / per_row);
        if (r >= std::min(N2, 8) || t == 2) rc = r;
    }
    if (rc < 1) return false;
    rc = std::min(rc, N2);
    const int chunks = (N2 + rc - 1) / rc;
    rc = (N2 + chunks - 1) / chunks;
    h->RC = rc;
    h->pd_smem = fixed + per_row * rc;
    const int r0 = h->pz.npass > 0 ? h->pz.radix[0] : 1;
    const int bf = rc * (N3 / r0);
    h->pd_threads = (int)align_up((size_t)std::min(256, std::max(64, bf)), 32);
    return true;
}

}  // namespace

extern "C" {

const char *rpa_last_error(void) { return g_err; }

size_t rpa_chi0_workspace_bytes(const int32_t grid[3], const double cell[9], const double q_red[3], double ecut_ha,
                                int32_t n_omega, int32_t max_batch_pairs, int32_t max_proj_total) {
    if (!valid_dims(grid, cell, q_red, ecut_ha, n_omega) || max_proj_total < 0 || max_proj_total > MAX_PROJ) {
        fail(RPA_ERR_INVALID_ARG, "rpa_chi0_workspace_bytes: invalid arguments");
        return 0;
    }
    double B[9], vol;
    recip_lattice(cell, B, &vol);
    if (!(vol > 0.0)) {
        fail(RPA_ERR_INVALID_ARG, "rpa_chi0_workspace_bytes: singular cell");
        return 0;
    }
    Sphere sp;
    build_sphere(grid, B, q_red, ecut_ha, &sp);
    if (sp.ng < 1) {
        fail(RPA_ERR_INVALID_ARG, "rpa_chi0_workspace_bytes: empty sphere");
        return 0;
    }
    Layout L;
    make_layout(grid, sp, n_omega, max_batch_pairs, max_proj_total, &L);
    return L.total;
}

}  // extern "C"

namespace {
// eta < 0: imaginary axis (n_freq slots); eta > 0: real axis (2 n_freq slots, omega of any sign)
int create_impl(rpa_chi0_t **out, const int32_t grid[3], const double cell[9], const double q_red[3], double ecut_ha,
                int32_t n_freq, const double *omega_ha, const double *omega_wt, double eta, int32_t max_batch_pairs,
                int32_t max_proj_total, void *workspace, size_t workspace_bytes, void *cuda_stream) {
    if (!out) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_create: out is NULL");
    *out = nullptr;
    if (!valid_dims(grid, cell, q_red, ecut_ha, n_freq) || !omega_ha || max_proj_total < 0 || max_proj_total > MAX_PROJ ||
        n_freq > (1 << 20))
        return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_create: invalid arguments");
    const bool real_axis = eta > 0.0;
    for (int i = 0; i < n_freq; i++) {
        if (real_axis ? !std::isfinite(omega_ha[i]) : !(omega_ha[i] > 0.0))
            return fail(RPA_ERR_INVALID_ARG, real_axis ? "rpa_chi0_create_real_axis: omega[%d] must be finite"
                                                       : "rpa_chi0_create: omega[%d] must be > 0", i);
    }
    const int n_omega = real_axis ? 2 * n_freq : n_freq;
    if (!workspace) return fail(RPA_ERR_WORKSPACE, "rpa_chi0_create: workspace is NULL");
    if (((uintptr_t)workspace & 255) != 0) return fail(RPA_ERR_WORKSPACE, "rpa_chi0_create: workspace not 256-byte aligned");

    rpa_chi0 *h = new (std::nothrow) rpa_chi0();
    if (!h) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_create: out of host memory");
    h->stream = (cudaStream_t)cuda_stream;
    memcpy(h->grid, grid, sizeof(h->grid));
    memcpy(h->cell, cell, sizeof(h->cell));
    memcpy(h->q, q_red, sizeof(h->q));
    h->ecut = ecut_ha;
    recip_lattice(cell, h->B, &h->vol);
    if (!(h->vol > 0.0)) { delete h; return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_create: singular cell"); }
    h->n_omega = n_omega;
    h->n_freq = n_freq;
    h->eta = real_axis ? eta : -1.0;
    h->omega.resize(n_omega);
    for (int i = 0; i < n_omega; i++) h->omega[i] = omega_ha[real_axis ? i / 2 : i];
    h->has_wt = omega_wt != nullptr && !real_axis;
    if (h->has_wt) h->wt.assign(omega_wt, omega_wt + n_omega);
    else h->wt.assign(n_omega, 0.0);
    build_sphere(grid, h->B, q_red, ecut_ha, &h->sp);
    if (h->sp.ng < 1) { delete h; return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_create: empty sphere"); }
    if (!fft_make_plan(grid[2], &h->pz) || !fft_make_plan(grid[1], &h->py)) {
        delete h;
        return fail(RPA_ERR_UNSUPPORTED, "rpa_chi0_create: grid lengths N2, N3 must factor into 2, 3, 5, 7");
    }
    h->max_proj = max_proj_total;
    make_layout(grid, h->sp, n_omega, max_batch_pairs, max_proj_total, &h->L);
    if (workspace_bytes < h->L.total) {
        const size_t need = h->L.total;
        delete h;
        return fail(RPA_ERR_WORKSPACE, "rpa_chi0_create: workspace %zu B < required %zu B", workspace_bytes, need);
    }
    h->ws = (unsigned char *)workspace;
    h->q0 = q_red[0] == 0.0 && q_red[1] == 0.0 && q_red[2] == 0.0;
    if (h->q0) {
        for (int s = 0; s < h->sp.ng; s++)
            if (h->sp.g[3 * s] == 0 && h->sp.g[3 * s + 1] == 0 && h->sp.g[3 * s + 2] == 0) h->idx0 = s;
        if (h->idx0 < 0) { delete h; return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_create: q = 0 but G = 0 is outside the sphere"); }
    }
    const bool pd_ok = plan_plane_kernel(h);
    if (!pd_ok && !h->zy_kernel) {
        delete h;
        return fail(RPA_ERR_UNSUPPORTED, "rpa_chi0_create: grid plane too large for shared memory");
    }

#define CREATE_TRY(expr)                                                                        \
    do {                                                                                        \
        cudaError_t e_ = (expr);                                                                \
        if (e_ != cudaSuccess) {                                                                \
            delete h;                                                                           \
            return fail(RPA_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_));                 \
        }                                                                                       \
    } while (0)

    if (pd_ok) CREATE_TRY(cudaFuncSetAttribute(h->pd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->pd_smem));
    {
        const size_t xs = (size_t)grid[0] * PD_G1_BLOCK * sizeof(cd);   // DFT table of pd_xaxis_kernel
        if (xs > 220 * 1024) { delete h; return fail(RPA_ERR_UNSUPPORTED, "rpa_chi0_create: N1 = %d too large for the x-axis table", grid[0]); }
        if (xs > 48 * 1024) CREATE_TRY(cudaFuncSetAttribute(pd_xaxis_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)xs));
    }
    {
        int dev = 0;
        CREATE_TRY(cudaGetDevice(&dev));
        CREATE_TRY(cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, dev));
        // highest priority: the block scheduler then places the (small) panel grids as soon as slots free up, instead
        // of after the last CTA of the trailing update in flight has been dispatched
        int prio_lo = 0, prio_hi = 0;
        CREATE_TRY(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
        CREATE_TRY(cudaStreamCreateWithPriority(&h->side, cudaStreamNonBlocking, prio_hi));
        for (cudaEvent_t *e : {&h->ev_panel[0], &h->ev_panel[1], &h->ev_col, &h->ev_fork})
            CREATE_TRY(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
        for (int l = 0; l < EC_MAX_LANES - 1; l++) {
            CREATE_TRY(cudaStreamCreateWithPriority(&h->xside[l], cudaStreamNonBlocking, prio_hi));
            CREATE_TRY(cudaStreamCreateWithPriority(&h->xmain[l], cudaStreamNonBlocking, prio_lo));
            for (cudaEvent_t *e : {&h->xev_panel[l][0], &h->xev_panel[l][1], &h->xev_col[l], &h->xev_join[l]})
                CREATE_TRY(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
        }
    }
    if (h->zy_kernel) {
        CREATE_TRY(cudaFuncSetAttribute(h->zy_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->zy_smem));
        int per_sm = 0;
        CREATE_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, h->zy_kernel, h->zy_threads, h->zy_smem));
        if (per_sm < 1) { delete h; return fail(RPA_ERR_CUDA, "rpa_chi0_create: pd_zy kernel does not fit an SM"); }
        h->zy_ctas_per_sm = per_sm;
    }
    CREATE_TRY(cudaFuncSetAttribute(rank_k_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, rk::Cfg<true>::SMEM_BYTES));
    CREATE_TRY(cudaFuncSetAttribute(rank_k3m_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, rk3::SMEM_BYTES));
    {
        // tensor map of the N buffer ([pair][ldn] complex = [pair][2 ldn] doubles): the driver entry point is fetched through
        // the runtime, so the library links against nothing but cudart
        typedef CUresult (*EncodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                        const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                        CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        CREATE_TRY(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
        if (!fn || qres != cudaDriverEntryPointSuccess) { delete h; return fail(RPA_ERR_CUDA, "rpa_chi0_create: cuTensorMapEncodeTiled unavailable"); }
        const cuuint64_t gdim[2] = {(cuuint64_t)(2 * h->L.ldn), (cuuint64_t)h->L.Kmax};
        const cuuint64_t gstride[1] = {(cuuint64_t)(h->L.ldn * sizeof(cd))};
        const cuuint32_t box[2] = {(cuuint32_t)rk3::BOX_DOUBLES, (cuuint32_t)rk3::KC};
        const cuuint32_t estr[2] = {1, 1};
        const CUresult cr = ((EncodeTiled)fn)(&h->nmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, h->ws + h->L.Nbuf, gdim, gstride, box, estr,
                                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (cr != CUDA_SUCCESS) { delete h; return fail(RPA_ERR_CUDA, "rpa_chi0_create: cuTensorMapEncodeTiled failed (%d)", (int)cr); }
        const cuuint64_t sdim[2] = {(cuuint64_t)h->L.ldn, (cuuint64_t)h->L.Kmax};
        const cuuint64_t sstride[1] = {(cuuint64_t)(h->L.ldn * sizeof(double))};
        const cuuint32_t sbox[2] = {(cuuint32_t)rk3::SBOX_DOUBLES, (cuuint32_t)rk3::KC};
        const CUresult cs = ((EncodeTiled)fn)(&h->smap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, h->ws + h->L.NS, sdim, sstride, sbox, estr,
                                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (cs != CUDA_SUCCESS) { delete h; return fail(RPA_ERR_CUDA, "rpa_chi0_create: cuTensorMapEncodeTiled (row sums) failed (%d)", (int)cs); }
    }
    // the chi0 accumulation runs on the FP64 tensor cores (rank_k3m_kernel) unless rpa_chi0_set_rank_k_mode says otherwise
    CREATE_TRY(cudaFuncSetAttribute(rank_k_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, rk::Cfg<false>::SMEM_BYTES));
    CREATE_TRY(cudaFuncSetAttribute(chol_update32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, cu32::smem_bytes(CH_P * CH_NB)));

    // tables: twiddles in extended precision, box -> sphere map
    const Sphere &sp = h->sp;
    const Layout &L = h->L;
    std::vector<cd> tw;
    const size_t twoff[3] = {L.tw1, L.tw2, L.tw3};
    for (int d = 0; d < 3; d++) {
        const int n = grid[d];
        tw.resize(n);
        for (int t = 0; t < n; t++) {
            const long double ang = -2.0L * 3.14159265358979323846264338327950288L * (long double)t / (long double)n;
            tw[t] = make_double2((double)cosl(ang), (double)sinl(ang));
        }
        CREATE_TRY(cudaMemcpyAsync(h->ws + twoff[d], tw.data(), n * sizeof(cd), cudaMemcpyHostToDevice, h->stream));
        CREATE_TRY(cudaStreamSynchronize(h->stream));
    }
    const int ng1 = sp.gmax[0] - sp.gmin[0] + 1, ng2 = sp.gmax[1] - sp.gmin[1] + 1, ng3 = sp.gmax[2] - sp.gmin[2] + 1;
    // (x frequency, kept column) -> sphere index or -1
    std::vector<int32_t> colof((size_t)ng2 * ng3, -1);
    for (int c = 0; c < sp.ncols; c++) colof[(size_t)(sp.coltab[c] >> 16) * ng3 + (sp.coltab[c] & 0xffff)] = c;
    std::vector<int32_t> box2s((size_t)ng1 * sp.ncols, -1);
    for (int s = 0; s < sp.ng; s++) {
        const int a = sp.g[3 * s] - sp.gmin[0], b = sp.g[3 * s + 1] - sp.gmin[1], c = sp.g[3 * s + 2] - sp.gmin[2];
        box2s[(size_t)a * sp.ncols + colof[(size_t)b * ng3 + c]] = s;
    }
    CREATE_TRY(cudaMemcpyAsync(h->ws + L.box2s, box2s.data(), box2s.size() * sizeof(int32_t), cudaMemcpyHostToDevice, h->stream));
    CREATE_TRY(cudaMemcpyAsync(h->ws + L.coltab, sp.coltab.data(), sp.coltab.size() * sizeof(int32_t), cudaMemcpyHostToDevice, h->stream));
    CREATE_TRY(cudaMemcpyAsync(h->ws + L.rowtab, sp.rowtab.data(), sp.rowtab.size() * sizeof(int32_t), cudaMemcpyHostToDevice, h->stream));
    CREATE_TRY(cudaMemcpyAsync(h->ws + L.Kc, sp.Kc.data(), sp.Kc.size() * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    CREATE_TRY(cudaMemcpyAsync(h->ws + L.omega, h->omega.data(), n_omega * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    CREATE_TRY(cudaMemcpyAsync(h->ws + L.wt, h->wt.data(), n_omega * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    const std::vector<int32_t> rkorder = rk3_tile_order(sp.ng);
    CREATE_TRY(cudaMemcpyAsync(h->ws + L.rkorder, rkorder.data(), rkorder.size() * sizeof(int32_t), cudaMemcpyHostToDevice, h->stream));
    {
        std::vector<double> wneg((size_t)L.ec_group * CH_P * CH_NB, -1.0);   // weight of the Cholesky trailing update
        CREATE_TRY(cudaMemcpyAsync(h->ws + L.wneg, wneg.data(), wneg.size() * sizeof(double), cudaMemcpyHostToDevice, h->stream));
        CREATE_TRY(cudaStreamSynchronize(h->stream));
    }
    CREATE_TRY(cudaMemsetAsync(h->ws + L.Lt, 0, 2 * (size_t)L.ec_group * CH_P * CH_NB * L.ldn * sizeof(cd), h->stream));
    CREATE_TRY(cudaMemsetAsync(h->ws + L.S, 0, (size_t)n_omega * sp.ng * L.ldS * sizeof(cd), h->stream));
    CREATE_TRY(cudaMemsetAsync(h->ws + L.Nbuf, 0, (size_t)L.Kmax * L.ldn * sizeof(cd), h->stream));
    CREATE_TRY(cudaStreamSynchronize(h->stream));
#undef CREATE_TRY
    *out = h;
    return RPA_OK;
}
}  // namespace

extern "C" {

int rpa_chi0_create(rpa_chi0_t **out, const int32_t grid[3], const double cell[9], const double q_red[3],
                    double ecut_ha, int32_t n_omega, const double *omega_ha, const double *omega_wt,
                    int32_t max_batch_pairs, int32_t max_proj_total, void *workspace, size_t workspace_bytes,
                    void *cuda_stream) {
    return create_impl(out, grid, cell, q_red, ecut_ha, n_omega, omega_ha, omega_wt, -1.0, max_batch_pairs, max_proj_total,
                       workspace, workspace_bytes, cuda_stream);
}

int rpa_chi0_create_real_axis(rpa_chi0_t **out, const int32_t grid[3], const double cell[9], const double q_red[3],
                              double ecut_ha, int32_t n_omega, const double *omega_ha, double eta_ha,
                              int32_t max_batch_pairs, int32_t max_proj_total, void *workspace, size_t workspace_bytes,
                              void *cuda_stream) {
    if (out) *out = nullptr;
    if (!(eta_ha > 0.0) || !std::isfinite(eta_ha))
        return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_create_real_axis: eta must be finite and > 0");
    return create_impl(out, grid, cell, q_red, ecut_ha, n_omega, omega_ha, nullptr, eta_ha, max_batch_pairs, max_proj_total,
                       workspace, workspace_bytes, cuda_stream);
}

int rpa_chi0_ng(const rpa_chi0_t *h, int32_t *ng) {
    if (!h || !ng) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_ng: NULL argument");
    *ng = h->sp.ng;
    return RPA_OK;
}

int rpa_chi0_gvectors(const rpa_chi0_t *h, int32_t *g, double *K2) {
    if (!h || !g) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_gvectors: NULL argument");
    memcpy(g, h->sp.g.data(), h->sp.g.size() * sizeof(int32_t));
    if (K2) memcpy(K2, h->sp.K2.data(), h->sp.K2.size() * sizeof(double));
    return RPA_OK;
}

}  // extern "C"

namespace {
// One batch of the chi0 accumulation on the int8 tensor cores (rank_k_i8.cuh): slicing passes + rank_k_i8_kernel<S> for
// every group of frequencies whose digit planes fit the scratch.  *done = false (nothing enqueued) when the batch cannot
// take this path: the exactness bound S K' 64^2 < 2^31 of the s32 accumulators does not hold (K' = 2 Kpad), the scratch
// is too small for one frequency, or there are more than RKI8_MAXW slots -- the caller then runs the FP64 tensor kernel.
template <int S>
int i8_batch(rpa_chi0 *h, int K, int Kpad, bool *done) {
    *done = false;
    const Layout &L = h->L;
    const int ng = h->sp.ng;
    cudaStream_t st = h->stream;
    if ((int64_t)S * 2 * Kpad * 4096 >= ((int64_t)1 << 31)) return RPA_OK;   // s32 accumulators could overflow: not error-free
    if (h->n_omega > RKI8_MAXW) return RPA_OK;
    cd *Nbuf = h->ptr<cd>(L.Nbuf);
    double *w = h->ptr<double>(L.w);
    // scratch (the pair-density buffer I is free again): invL | invR | tiles | PL | PR of a frequency group
    const int ngp = (ng + rki8::RB - 1) / rki8::RB * rki8::RB, nrb = 2 * ngp / rki8::RB;
    const int ncb = (ng + rki8::CB - 1) / rki8::CB, nkb = 2 * Kpad / rki8::KB, nt = (int)h->i8_tiles.size();
    const size_t scratch = (size_t)L.sub_pairs * L.I_pair_bytes;
    size_t off = 0;
    auto carve = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
    const size_t o_invL = carve((size_t)(1 + h->n_omega) * ngp * 8), o_invR = o_invL + (size_t)ngp * 8;
    const size_t o_tiles = carve((size_t)nt * sizeof(int2));
    const size_t o_PL = carve((size_t)nrb * nkb * S * rki8::A_BYTES);
    const size_t per_w = (size_t)ncb * nkb * S * rki8::B_BYTES;
    int wg = off < scratch ? (int)std::min<size_t>((size_t)h->n_omega, (scratch - off) / per_w) : 0;
    if (wg < 1) return RPA_OK;
    const int ngroups = (h->n_omega + wg - 1) / wg;
    wg = (h->n_omega + ngroups - 1) / ngroups;   // equal groups
    unsigned char *base = h->ws + L.I;
    double *invL = (double *)(base + o_invL), *invR = (double *)(base + o_invR);
    int2 *d_tiles = (int2 *)(base + o_tiles);
    int8_t *PL = (int8_t *)(base + o_PL), *PR = (int8_t *)(base + off);
    CUDA_TRY(cudaMemcpyAsync(d_tiles, h->i8_tiles.data(), (size_t)nt * sizeof(int2), cudaMemcpyHostToDevice, st));
    const int nmx = (1 + h->n_omega) * ngp;
    CUDA_TRY(cudaMemsetAsync(invL, 0, (size_t)nmx * 8, st));
    rki8_rowmax_kernel<<<dim3((ng + 127) / 128, std::max(1, std::min(64, K / 64))), 128, 0, st>>>(
        Nbuf, L.ldn, K, ng, w, L.ldw, h->n_omega, ngp, (unsigned long long *)invL);
    rki8_scale_finish_kernel<<<(nmx + 255) / 256, 256, 0, st>>>((unsigned long long *)invL, nmx);
    rki8_pack_left_kernel<S><<<dim3(nkb, nrb), 128, 0, st>>>(Nbuf, L.ldn, Kpad, ng, ngp, invL, PL);
    h->launches += 3;
    for (int iw0 = 0; iw0 < h->n_omega; iw0 += wg) {
        const int nw = std::min(wg, h->n_omega - iw0);
        const double *w0 = w + (size_t)iw0 * L.ldw, *invR0 = invR + (size_t)iw0 * ngp;
        cd *S0 = h->ptr<cd>(L.S) + (size_t)iw0 * ng * L.ldS;
        rki8_pack_right_kernel<S><<<dim3(nkb, ncb), 64, 0, st>>>(Nbuf, L.ldn, Kpad, ng, ngp, w0, L.ldw, nw, invR0, PR);
        StageTimer tm5(h, 5, 1);
        CUDA_TRY(launch_i8<S>(h->i8_cluster, dim3(nt, nw), st, PL, PR, nkb, ncb, d_tiles, invL, invR0, ng, ngp, S0, L.ldS,
                              (int64_t)ng * L.ldS));
        h->launches += 1;
    }
    h->launches -= 1;   // the caller's stage timer counts one
    *done = true;
    return RPA_OK;
}
}  // namespace

namespace {
#define ADD_ARGS_LOCALS                                                                                                  \
    const double kweight = A.kweight; const int32_t n_occ = A.n_occ, n_unocc = A.n_unocc, n_atoms = A.n_atoms;            \
    const void *psi_occ = A.psi_occ, *psi_unocc = A.psi_unocc, *P_occ = A.P_occ, *P_unocc = A.P_unocc, *Q = A.Q, *grad = A.grad; \
    const double *eps_occ = A.eps_occ, *eps_unocc = A.eps_unocc, *f_occ = A.f_occ, *f_unocc = A.f_unocc, *R_cart = A.R_cart, *qdir = A.qdir; \
    const int32_t *n_proj = A.n_proj;                                                                                    \
    (void)kweight; (void)n_occ; (void)n_unocc; (void)n_atoms; (void)psi_occ; (void)psi_unocc; (void)P_occ; (void)P_unocc; (void)Q; \
    (void)grad; (void)eps_occ; (void)eps_unocc; (void)f_occ; (void)f_unocc; (void)R_cart; (void)qdir; (void)n_proj;     \
    const Layout &L = h->L; const Sphere &sp = h->sp; const int ng = sp.ng; cudaStream_t st = h->stream;                 \
    (void)L; (void)sp; (void)ng; (void)st

// validation, PAW metadata and band energies / occupations to the device; *ptot_out = sum of n_proj.
// Returns 1 (not an error code) when the band set is empty: nothing to add.
int add_setup(rpa_chi0_t *h, const AddArgs &A, int *ptot_out) {
    if (!h) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint: handle is NULL");
    if (h->q0 && !A.grad)
        return fail(RPA_ERR_UNSUPPORTED, "rpa_chi0_add_kpoint: the handle has q = 0: use rpa_chi0_add_kpoint_optical (P:L113-134)");
    if (!h->q0 && A.grad) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint_optical: the handle has q != 0");
    if (A.n_occ < 0 || A.n_unocc < 0 || A.n_atoms < 0) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint: negative count");
    if (A.n_occ == 0 || A.n_unocc == 0) return 1;  // empty band set: nothing to add
    if (!A.psi_occ || !A.psi_unocc || !A.eps_occ || !A.eps_unocc || !A.f_occ || !A.f_unocc)
        return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint: NULL band array");
    if ((int64_t)A.n_occ + A.n_unocc > MAX_BANDS) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint: more than %d bands", MAX_BANDS);
    ADD_ARGS_LOCALS;

    // ---- PAW metadata ----------------------------------------------------------------------------------
    int ptot = 0;
    if (n_atoms > 0) {
        if (!n_proj || !P_occ || !P_unocc || !Q || !R_cart) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint: NULL PAW array");
        if (n_atoms > MAX_ATOMS) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint: more than %d atoms", MAX_ATOMS);
        std::vector<int32_t> aj_atom, aj_j, poff(n_atoms), ni(n_atoms);
        std::vector<int64_t> qoff(n_atoms);
        int64_t qo = 0;
        for (int a = 0; a < n_atoms; a++) {
            if (n_proj[a] < 0) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint: n_proj[%d] < 0", a);
            poff[a] = ptot;
            ni[a] = n_proj[a];
            qoff[a] = qo;
            for (int j = 0; j < n_proj[a]; j++) { aj_atom.push_back(a); aj_j.push_back(j); }
            ptot += n_proj[a];
            qo += (int64_t)n_proj[a] * n_proj[a] * ng;
        }
        if (ptot > h->max_proj)
            return fail(RPA_ERR_WORKSPACE, "rpa_chi0_add_kpoint: %d projectors > max_proj_total %d given at create", ptot, h->max_proj);
        if (ptot > 0) {
            CUDA_TRY(cudaMemcpyAsync(h->ws + L.aj_atom, aj_atom.data(), ptot * sizeof(int32_t), cudaMemcpyHostToDevice, st));
            CUDA_TRY(cudaMemcpyAsync(h->ws + L.aj_j, aj_j.data(), ptot * sizeof(int32_t), cudaMemcpyHostToDevice, st));
            CUDA_TRY(cudaMemcpyAsync(h->ws + L.atom_poff, poff.data(), n_atoms * sizeof(int32_t), cudaMemcpyHostToDevice, st));
            CUDA_TRY(cudaMemcpyAsync(h->ws + L.atom_ni, ni.data(), n_atoms * sizeof(int32_t), cudaMemcpyHostToDevice, st));
            CUDA_TRY(cudaMemcpyAsync(h->ws + L.atom_qoff, qoff.data(), n_atoms * sizeof(int64_t), cudaMemcpyHostToDevice, st));
            CUDA_TRY(cudaMemcpyAsync(h->ws + L.R, R_cart, (size_t)n_atoms * 3 * sizeof(double), cudaMemcpyHostToDevice, st));
            // the vectors above are pageable host memory: the copies have been staged when the calls return
        }
    }
    double *band = h->ptr<double>(L.band);
    double *d_eo = band, *d_fo = band + n_occ, *d_eu = band + 2 * (size_t)n_occ, *d_fu = band + 2 * (size_t)n_occ + n_unocc;
    CUDA_TRY(cudaMemcpyAsync(d_eo, eps_occ, n_occ * sizeof(double), cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(d_fo, f_occ, n_occ * sizeof(double), cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(d_eu, eps_unocc, n_unocc * sizeof(double), cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(d_fu, f_unocc, n_unocc * sizeof(double), cudaMemcpyHostToDevice, st));

    *ptot_out = ptot;
    return RPA_OK;
}

// S2 + S3 (pair product, pruned 3-D FFT, sphere gather) of the pairs [p0, p0 + pc) of a batch (pair p: band n = n0 + p / mlen,
// m = m0 + p % mlen) into rows p0 ... of the N buffer; pc <= L.sub_pairs.  win: the rows of the N buffer when the pairs are a window of a
// larger batch (PdRowWindow, pair_density.cuh).
int add_pair_densities(rpa_chi0_t *h, const AddArgs &A, int n0, int mlen, int m0, int p0, int pc,
                       PdRowWindow win = PdRowWindow{INT_MAX, 0, 0}) {
    ADD_ARGS_LOCALS;
    const int N1 = h->grid[0], N2 = h->grid[1], N3 = h->grid[2];
    const int ng1 = sp.gmax[0] - sp.gmin[0] + 1, ng2 = sp.gmax[1] - sp.gmin[1] + 1, ng3 = sp.gmax[2] - sp.gmin[2] + 1;
    const double inv_n = 1.0 / ((double)N1 * N2 * N3);
    cd *Nbuf = h->ptr<cd>(L.Nbuf);
    (void)N2; (void)N3;
    if (h->zy_kernel) {
        StageTimer tm(h, 0, 1);
        PdZyParams P;
        P.psi_occ = (const cd *)psi_occ; P.psi_unocc = (const cd *)psi_unocc;
        P.I = h->ptr<cd>(L.I);
        P.coltab = h->ptr<int32_t>(L.coltab); P.rowtab = h->ptr<int32_t>(L.rowtab); P.ncols = sp.ncols;
        P.tw3 = h->ptr<cd>(L.tw3); P.tw2 = h->ptr<cd>(L.tw2);
        P.N1 = N1;
        P.n0 = n0; P.mlen = mlen; P.m0 = m0;
        P.p_begin = p0; P.p_count = pc;
        pdzy_plan_units(P, h->zy_G);
        P.g2min = sp.gmin[1]; P.ng2 = ng2; P.g3min = sp.gmin[2]; P.ng3 = ng3;
        // persistent 1-D grid: one CTA per resident slot, work items (unit, plane) dealt round-robin
        const int nctas = std::max(1, std::min(P.n_units * N1, h->n_sm * h->zy_ctas_per_sm));
        h->zy_kernel<<<nctas, h->zy_threads, h->zy_smem, st>>>(P);
        CUDA_TRY(cudaGetLastError());
    } else {
        StageTimer tm(h, 0, 1);
        PdPlaneParams P;
        P.psi_occ = (const cd *)psi_occ; P.psi_unocc = (const cd *)psi_unocc;
        P.I = h->ptr<cd>(L.I);
        P.coltab = h->ptr<int32_t>(L.coltab); P.ncols = sp.ncols;
        P.tw3 = h->ptr<cd>(L.tw3); P.tw2 = h->ptr<cd>(L.tw2);
        P.N1 = N1; P.N2 = N2; P.N3 = N3;
        P.n0 = n0; P.mlen = mlen; P.m0 = m0;
        P.p_begin = p0; P.p_count = pc;
        P.g2min = sp.gmin[1]; P.ng2 = ng2; P.g3min = sp.gmin[2]; P.ng3 = ng3;
        P.RC = h->RC; P.nbuf = h->pd_nbuf; P.pz = h->pz; P.py = h->py;
        const int gy = std::max(1, std::min(pc, (148 * 8 + N1 - 1) / N1));
        h->pd_kernel<<<dim3(N1, gy), h->pd_threads, h->pd_smem, st>>>(P);
        CUDA_TRY(cudaGetLastError());
    }
    {
        StageTimer tm(h, 1, 1);
        const int xslots = pd_xaxis8_slots(N1, sp.gmin[0], ng1);
        const int ncols = sp.ncols;   // the x transform runs on the kept (g2, g3) columns only
        const int xth = std::min(128, (ncols + 31) / 32 * 32);   // 73 kept columns (configs[2]): 96 threads, not 128
        const int xbx = (ncols + xth - 1) / xth;
        // short x axes (compile-time N1): blocks walk over the pairs, as many as keep every SM busy with ~8 blocks;
        // long axes: one block per (column block, pair) as before (measured: the walk loses 4-5 % there)
        const bool xshort = xslots == 2 && (N1 == 24 || N1 == 16);
        int xby = pc;
        if (xshort) {
            // every block resident at once and the same number of pairs for each: ceil(pc xbx / slots) rounds of
            // the pair loop (2400 pairs of a configs[2] k-point on 740 slots: 600 blocks x 4 pairs, not 1184 x 2-3 in
            // two waves)
            int per_sm = 0;
            const void *xk = N1 == 24 ? (const void *)pd_xaxis8_kernel<2, 3> : (const void *)pd_xaxis8_kernel<2, 2>;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, xk, xth, (size_t)N1 * 2 * sizeof(cd)) != cudaSuccess || per_sm < 1)
                per_sm = 4;
            const int slots = std::max(1, h->n_sm * per_sm / xbx);
            const int rounds = (pc + slots - 1) / slots;
            xby = (pc + rounds - 1) / rounds;
        }
#define X8_ARGS h->ptr<cd>(L.I), Nbuf, L.ldn, h->ptr<cd>(L.tw1), h->ptr<int32_t>(L.box2s), N1, ncols, sp.gmin[0], ng1, p0, pc, inv_n, win
        if (xslots == 2 && N1 == 24)
            pd_xaxis8_kernel<2, 3><<<dim3(xbx, xby), xth, (size_t)N1 * 2 * sizeof(cd), st>>>(X8_ARGS);
        else if (xslots == 2 && N1 == 16)
            pd_xaxis8_kernel<2, 2><<<dim3(xbx, xby), xth, (size_t)N1 * 2 * sizeof(cd), st>>>(X8_ARGS);
        else if (xslots == 2)
            pd_xaxis8_kernel<2, 0><<<dim3(xbx, xby), xth, (size_t)N1 * 2 * sizeof(cd), st>>>(X8_ARGS);
        else if (xslots == 3)
            pd_xaxis8_kernel<3, 0><<<dim3(xbx, xby), xth, (size_t)N1 * 3 * sizeof(cd), st>>>(X8_ARGS);
#undef X8_ARGS
        else
            pd_xaxis_kernel<<<dim3((ncols + 127) / 128, pc), 128, (size_t)N1 * PD_G1_BLOCK * sizeof(cd), st>>>(
                h->ptr<cd>(L.I), Nbuf, L.ldn, h->ptr<cd>(L.tw1), h->ptr<int32_t>(L.box2s), N1, ncols, sp.gmin[0], ng1, p0, inv_n, win);
        CUDA_TRY(cudaGetLastError());
    }
    return RPA_OK;
}

// the rest of a batch of K = nslots mlen pairs whose pair densities are in the N buffer: S4 PAW, the optical head, S5 weights,
// S6 rank-K update of every frequency
int add_finish_batch(rpa_chi0_t *h, const AddArgs &A, int ptot, int n0, int nslots, int mlen, int m0) {
    ADD_ARGS_LOCALS;
    const int K = nslots * mlen;
    const int Kpad = (int)align_up((size_t)K, K_ALIGN);
    cd *Nbuf = h->ptr<cd>(L.Nbuf);
    double *w = h->ptr<double>(L.w);
    double *band = h->ptr<double>(L.band);
    double *d_eo = band, *d_fo = band + n_occ, *d_eu = band + 2 * (size_t)n_occ, *d_fu = band + 2 * (size_t)n_occ + n_unocc;
    // S4: PAW
    if (ptot > 0) {
        StageTimer tm(h, 2, 2);
        paw_T_kernel<<<dim3((ng + 127) / 128, ptot, nslots), 128, 0, st>>>(
            h->ptr<cd>(L.T), L.ldn, ng, ptot, (const cd *)P_occ, n0, (const cd *)Q, h->ptr<int32_t>(L.aj_atom),
            h->ptr<int32_t>(L.aj_j), h->ptr<int32_t>(L.atom_poff), h->ptr<int32_t>(L.atom_ni),
            h->ptr<int64_t>(L.atom_qoff), h->ptr<double>(L.R), h->ptr<double>(L.Kc));
        CUDA_TRY(cudaGetLastError());
        const int chunks = (mlen + PAW_PB - 1) / PAW_PB;
        paw_add_kernel<<<dim3((ng + 127) / 128, nslots * chunks), 128, 0, st>>>(
            Nbuf, L.ldn, ng, ptot, h->ptr<cd>(L.T), (const cd *)P_unocc, mlen, m0);
        CUDA_TRY(cudaGetLastError());
    }
    // step 10: optical limit, the G = 0 element of every pair density of the batch
    if (grad) {
        optical_head_kernel<<<(K + 127) / 128, 128, 0, st>>>(Nbuf, L.ldn, h->idx0, K, n0, mlen, m0, n_occ, n_unocc, d_eo,
                                                            d_eu, qdir[0], qdir[1], qdir[2], (const cd *)grad);
        h->launches += 1;
        CUDA_TRY(cudaGetLastError());
    }
    // S5: weights
    {
        StageTimer tm(h, 3, 1);
        weights_kernel<<<dim3((Kpad + 127) / 128, h->n_omega), 128, 0, st>>>(
            w, L.ldw, K, Kpad, h->ptr<double>(L.omega), h->n_omega, d_eo, d_fo, d_eu, d_fu, n0, mlen, m0, kweight, h->eta);
        CUDA_TRY(cudaGetLastError());
    }
    // S6: rank-K update of every frequency
    {
        StageTimer tm(h, 4, 1);
        bool done_i8 = false;
        if (h->use_i8 && (h->i8_force || (ng >= I8_MIN_NG && K >= I8_MIN_K))) {
            int rc = RPA_OK;
            switch (h->i8_digits) {
                case 6: rc = i8_batch<6>(h, K, Kpad, &done_i8); break;
                case 8: rc = i8_batch<8>(h, K, Kpad, &done_i8); break;
                default: rc = i8_batch<7>(h, K, Kpad, &done_i8); break;
            }
            if (rc != RPA_OK) return rc;
        }
        (done_i8 ? h->i8_batches : h->fp64_batches) += 1;
        if (done_i8) {
        } else if (h->use_3m) {
            // whole waves (one CTA per SM) with full K, then the last partial wave K-sliced so that it fills the GPU too
            const int ntiles = ntiles_lower(ng, rk3::T), units = ntiles * h->n_omega, nchunks = Kpad / rk3::KC;
            const int whole = units / h->n_sm * h->n_sm;
            const int tail = units - whole;
            auto launch = [&](int off, int count, int ksplit) {
                rank_k3m_kernel<<<dim3(count, 1, ksplit), rk3::THREADS, rk3::SMEM_BYTES, st>>>(
                    h->nmap, h->smap, Kpad, w, L.ldw, h->ptr<cd>(L.S), L.ldS, (int64_t)ng * L.ldS, ng, h->n_omega, off, h->ptr<int32_t>(L.rkorder));
            };
            // third operand plane of the 3M product: NS = Re N + Im N, one pass over the batch's N
            rk3_rowsum_kernel<<<dim3(Kpad, (unsigned)((L.ldn + 255) / 256)), 256, 0, st>>>(Nbuf, L.ldn, h->ptr<double>(L.NS));
            h->launches += 1;
            double c_single = 0.0, c_tail = 0.0;
            const int s_single = pick_ksplit(units, nchunks, h->n_sm, &c_single, 512 / rk3::KC);
            const int s_tail = tail > 0 ? pick_ksplit(tail, nchunks, h->n_sm, &c_tail, 512 / rk3::KC) : 1;
            // two launches only if the model says they save at least a tenth of an item, and only behind at least eight waves:
            // the first launch ends ragged (tiles differ in work) and the second waits for its last CTA, which on the three
            // waves of configs[2] costs more than the sliced remainder saves (0.871 against 0.781 ms per k-point)
            if (whole >= 8 * h->n_sm && tail > 0 && whole / h->n_sm + c_tail + 0.1 < c_single) {
                launch(0, whole, 1);
                launch(whole, tail, s_tail);
                h->launches += 1;
            } else {
                launch(0, units, s_single);
            }
        } else {
            const int units = ntiles_lower(ng, rk::T) * ((h->n_omega + rk::Cfg<true>::NW - 1) / rk::Cfg<true>::NW);
            const int ksplit = pick_ksplit(units, Kpad / rk::KC, h->n_sm);
            rank_k_kernel<true><<<dim3(ntiles_lower(ng, rk::T), (h->n_omega + rk::Cfg<true>::NW - 1) / rk::Cfg<true>::NW, ksplit),
                                  rk::Cfg<true>::THREADS, rk::Cfg<true>::SMEM_BYTES, st>>>(
                Nbuf, L.ldn, 0, Kpad, w, L.ldw, h->ptr<cd>(L.S), L.ldS, (int64_t)ng * L.ldS, ng, 0, h->n_omega, 0, ng);
        }
        CUDA_TRY(cudaGetLastError());
    }
    return RPA_OK;
}

// rows K ... Kpad of the N buffer must be zero (they meet zero weights, but 0 * NaN is NaN)
int add_zero_padding(rpa_chi0_t *h, int K) {
    const Layout &L = h->L;
    const int Kpad = (int)align_up((size_t)K, K_ALIGN);
    if (Kpad > K) CUDA_TRY(cudaMemsetAsync(h->ptr<cd>(L.Nbuf) + (size_t)K * L.ldn, 0, (size_t)(Kpad - K) * L.ldn * sizeof(cd), h->stream));
    return RPA_OK;
}

// batches of a call: either several whole occupied rows, or a slice of one row
void add_batching(const rpa_chi0_t *h, int n_unocc, int *rows_per_batch, int *mchunk) {
    const int Kmax = h->L.Kmax;
    *rows_per_batch = 1;
    *mchunk = n_unocc;
    if (n_unocc >= Kmax) {
        const int nch = (n_unocc + Kmax - 1) / Kmax;
        *mchunk = std::min((int)align_up((size_t)(n_unocc + nch - 1) / nch, K_ALIGN), Kmax);
    } else {
        *rows_per_batch = std::max(1, std::min(MAX_SLOTS, Kmax / n_unocc));
    }
}

// rpa_chi0_add_kpoint, and rpa_chi0_add_kpoint_optical when grad != NULL (q = 0 handle: G = 0 element replaced)
int add_kpoint_impl(rpa_chi0_t *h, const AddArgs &A) {
    if (h && h->pend_open) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint: a streamed k-point is open (rpa_chi0_add_kpoint_end)");
    int ptot = 0;
    {
        const int rc = add_setup(h, A, &ptot);
        if (rc != RPA_OK) return rc == 1 ? RPA_OK : rc;
    }
    int rows_per_batch, mchunk;
    add_batching(h, A.n_unocc, &rows_per_batch, &mchunk);
    for (int n0 = 0; n0 < A.n_occ; n0 += rows_per_batch) {
        const int nslots = std::min(rows_per_batch, A.n_occ - n0);
        for (int m0 = 0; m0 < A.n_unocc; m0 += mchunk) {
            const int mlen = std::min(mchunk, A.n_unocc - m0);
            const int K = nslots * mlen;
            int rc = add_zero_padding(h, K);
            for (int p0 = 0; p0 < K && rc == RPA_OK; p0 += h->L.sub_pairs)
                rc = add_pair_densities(h, A, n0, mlen, m0, p0, std::min(h->L.sub_pairs, K - p0));
            if (rc == RPA_OK) rc = add_finish_batch(h, A, ptot, n0, nslots, mlen, m0);
            if (rc != RPA_OK) return rc;
        }
    }
    return RPA_OK;
}
}  // namespace

extern "C" {

int rpa_chi0_add_kpoint(rpa_chi0_t *h, double kweight, int32_t n_occ, const void *psi_occ, int32_t n_unocc,
                        const void *psi_unocc, const double *eps_occ, const double *eps_unocc, const double *f_occ,
                        const double *f_unocc, int32_t n_atoms, const int32_t *n_proj, const void *P_occ,
                        const void *P_unocc, const void *Q, const double *R_cart) {
    const AddArgs A = {kweight, n_occ, psi_occ, n_unocc, psi_unocc, eps_occ, eps_unocc, f_occ, f_unocc, n_atoms, n_proj,
                       P_occ, P_unocc, Q, R_cart, nullptr, nullptr};
    return add_kpoint_impl(h, A);
}

int rpa_chi0_add_kpoint_optical(rpa_chi0_t *h, double kweight, int32_t n_occ, const void *psi_occ, int32_t n_unocc,
                                const void *psi_unocc, const double *eps_occ, const double *eps_unocc, const double *f_occ,
                                const double *f_unocc, int32_t n_atoms, const int32_t *n_proj, const void *P_occ,
                                const void *P_unocc, const void *Q, const double *R_cart, const double qdir_cart[3],
                                const void *grad) {
    if (!qdir_cart || !grad) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint_optical: NULL direction or gradient");
    const double nrm = sqrt(qdir_cart[0] * qdir_cart[0] + qdir_cart[1] * qdir_cart[1] + qdir_cart[2] * qdir_cart[2]);
    if (!(nrm > 0.0) || !std::isfinite(nrm)) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint_optical: zero direction");
    const double qd[3] = {qdir_cart[0] / nrm, qdir_cart[1] / nrm, qdir_cart[2] / nrm};
    const AddArgs A = {kweight, n_occ, psi_occ, n_unocc, psi_unocc, eps_occ, eps_unocc, f_occ, f_unocc, n_atoms, n_proj,
                       P_occ, P_unocc, Q, R_cart, qd, grad};
    return add_kpoint_impl(h, A);
}

// rpa_chi0_add_kpoint in three steps, for unoccupied orbitals that are still being produced (include/rpa_chi0.h)
int rpa_chi0_add_kpoint_begin(rpa_chi0_t *h, double kweight, int32_t n_occ, const void *psi_occ, int32_t n_unocc,
                              const void *psi_unocc, const double *eps_occ, const double *eps_unocc, const double *f_occ,
                              const double *f_unocc, int32_t n_atoms, const int32_t *n_proj, const void *P_occ,
                              const void *P_unocc, const void *Q, const double *R_cart) {
    if (!h) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint_begin: handle is NULL");
    if (h->pend_open) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint_begin: the previous streamed k-point was not ended");
    if (n_occ < 1 || n_unocc < 1) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint_begin: empty band set");
    int rows_per_batch, mchunk;
    add_batching(h, n_unocc, &rows_per_batch, &mchunk);
    if (mchunk < n_unocc || n_occ > rows_per_batch)
        return fail(RPA_ERR_UNSUPPORTED, "rpa_chi0_add_kpoint_begin: %d x %d transitions are more than one batch (%d, at most %d occupied bands): use rpa_chi0_add_kpoint",
                    n_occ, n_unocc, h->L.Kmax, MAX_SLOTS);
    const AddArgs A = {kweight, n_occ, psi_occ, n_unocc, psi_unocc, eps_occ, eps_unocc, f_occ, f_unocc, n_atoms, n_proj,
                       P_occ, P_unocc, Q, R_cart, nullptr, nullptr};
    int ptot = 0;
    {
        const int rc = add_setup(h, A, &ptot);
        if (rc != RPA_OK) return rc;
    }
    {
        const int rc = add_zero_padding(h, n_occ * n_unocc);
        if (rc != RPA_OK) return rc;
    }
    h->pend = A;
    h->pend.eps_occ = h->pend.eps_unocc = h->pend.f_occ = h->pend.f_unocc = h->pend.R_cart = nullptr;   // consumed
    h->pend.n_proj = nullptr;
    h->pend_ptot = ptot;
    h->pend_m_next = 0;
    h->pend_open = true;
    return RPA_OK;
}

int rpa_chi0_add_kpoint_pairs(rpa_chi0_t *h, int32_t m_begin, int32_t m_end) {
    if (!h) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint_pairs: handle is NULL");
    if (!h->pend_open) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint_pairs: no streamed k-point is open");
    const AddArgs &A = h->pend;
    if (m_begin != h->pend_m_next || m_end < m_begin || m_end > A.n_unocc)
        return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint_pairs: bands [%d, %d): slices must follow one another from %d up to %d",
                    m_begin, m_end, h->pend_m_next, A.n_unocc);
    // the window as a batch of its own -- pair p' = n wl + j is (occupied band n, unoccupied band m_begin + j) -- whose pair
    // densities go to the rows n n_unocc + m_begin + j of the k-point's batch: one launch for all occupied bands
    const int wl = m_end - m_begin;
    if (wl > 0) {
        const PdRowWindow win = {wl, A.n_unocc, m_begin};
        const int K = A.n_occ * wl;
        for (int p0 = 0; p0 < K; p0 += h->L.sub_pairs) {
            const int rc = add_pair_densities(h, A, 0, wl, m_begin, p0, std::min(h->L.sub_pairs, K - p0), win);
            if (rc != RPA_OK) return rc;
        }
    }
    h->pend_m_next = m_end;
    return RPA_OK;
}

int rpa_chi0_add_kpoint_end(rpa_chi0_t *h) {
    if (!h) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint_end: handle is NULL");
    if (!h->pend_open) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint_end: no streamed k-point is open");
    h->pend_open = false;   // whatever happens below, the call is over
    if (h->pend_m_next != h->pend.n_unocc)
        return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_add_kpoint_end: only %d of %d unoccupied bands were given to rpa_chi0_add_kpoint_pairs; nothing added",
                    h->pend_m_next, h->pend.n_unocc);
    return add_finish_batch(h, h->pend, h->pend_ptot, 0, h->pend.n_occ, h->pend.n_unocc, 0);
}

// Eq. 15 / Eq. 19: gradient matrix elements between occupied and unoccupied bands given on a common plane-wave set.
int rpa_momentum_pw(rpa_chi0_t *h, const double k_cart[3], int32_t n_pw, const int32_t *g_pw, int32_t n_occ, const void *C_occ,
                    int32_t n_unocc, const void *C_unocc, int32_t n_atoms, const int32_t *n_proj, const void *P_occ,
                    const void *P_unocc, const void *Qgrad, void *grad_out) {
    if (!h || !k_cart) return fail(RPA_ERR_INVALID_ARG, "rpa_momentum_pw: NULL argument");
    if (n_pw < 0 || n_occ < 0 || n_unocc < 0 || n_atoms < 0) return fail(RPA_ERR_INVALID_ARG, "rpa_momentum_pw: negative count");
    if (n_occ == 0 || n_unocc == 0) return RPA_OK;
    if (!grad_out || (n_pw > 0 && (!g_pw || !C_occ || !C_unocc))) return fail(RPA_ERR_INVALID_ARG, "rpa_momentum_pw: NULL array");
    const Layout &L = h->L;
    cudaStream_t st = h->stream;
    const size_t out_bytes = (size_t)3 * n_occ * n_unocc * sizeof(cd);
    if ((size_t)3 * n_pw * sizeof(double) > (size_t)L.sub_pairs * L.I_pair_bytes)
        return fail(RPA_ERR_WORKSPACE, "rpa_momentum_pw: %d plane waves do not fit the handle's scratch", n_pw);
    if (n_pw == 0) {
        CUDA_TRY(cudaMemsetAsync(grad_out, 0, out_bytes, st));
    } else {
        std::vector<double> Kc((size_t)3 * n_pw);
        for (int q = 0; q < n_pw; q++)
            for (int al = 0; al < 3; al++)
                Kc[(size_t)al * n_pw + q] = k_cart[al] + g_pw[3 * q] * h->B[al] + g_pw[3 * q + 1] * h->B[3 + al] + g_pw[3 * q + 2] * h->B[6 + al];
        double *d_Kc = h->ptr<double>(L.I);
        CUDA_TRY(cudaMemcpyAsync(d_Kc, Kc.data(), Kc.size() * sizeof(double), cudaMemcpyHostToDevice, st));
        CUDA_TRY(cudaStreamSynchronize(st));   // Kc is pageable host memory about to go out of scope
        momentum_pw_kernel<<<dim3(n_unocc, (n_occ + OPT_NB - 1) / OPT_NB), 128, 0, st>>>((const cd *)C_occ, (const cd *)C_unocc, d_Kc,
                                                                                      n_pw, n_occ, n_unocc, (cd *)grad_out);
        h->launches += 1;
        CUDA_TRY(cudaGetLastError());
    }
    if (n_atoms > 0) {
        if (!n_proj || !P_occ || !P_unocc || !Qgrad) return fail(RPA_ERR_INVALID_ARG, "rpa_momentum_pw: NULL PAW array");
        if (n_atoms > MAX_ATOMS) return fail(RPA_ERR_INVALID_ARG, "rpa_momentum_pw: more than %d atoms", MAX_ATOMS);
        std::vector<int32_t> poff(n_atoms), ni(n_atoms);
        int ptot = 0;
        for (int a = 0; a < n_atoms; a++) {
            if (n_proj[a] < 0) return fail(RPA_ERR_INVALID_ARG, "rpa_momentum_pw: n_proj[%d] < 0", a);
            poff[a] = ptot;
            ni[a] = n_proj[a];
            ptot += n_proj[a];
        }
        if (ptot > 0) {
            CUDA_TRY(cudaMemcpyAsync(h->ws + L.atom_poff, poff.data(), n_atoms * sizeof(int32_t), cudaMemcpyHostToDevice, st));
            CUDA_TRY(cudaMemcpyAsync(h->ws + L.atom_ni, ni.data(), n_atoms * sizeof(int32_t), cudaMemcpyHostToDevice, st));
            CUDA_TRY(cudaStreamSynchronize(st));
            momentum_paw_kernel<<<dim3((n_unocc + 127) / 128, n_occ, 3), 128, 0, st>>>(
                (cd *)grad_out, n_occ, n_unocc, ptot, n_atoms, h->ptr<int32_t>(L.atom_poff), h->ptr<int32_t>(L.atom_ni),
                (const cd *)P_occ, (const cd *)P_unocc, (const cd *)Qgrad);
            h->launches += 1;
            CUDA_TRY(cudaGetLastError());
        }
    }
    return RPA_OK;
}

int rpa_chi0_get(rpa_chi0_t *h, int32_t i_omega, void *chi0_out) {
    if (!h || !chi0_out) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_get: NULL argument");
    if (i_omega < 0 || i_omega >= h->n_freq) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_get: i_omega %d out of range", i_omega);
    const int ng = h->sp.ng;
    const int nt = (ng + 31) / 32;
    const size_t strideS = (size_t)ng * h->L.ldS;
    if (h->eta > 0.0)
        chi0_get_real_axis_kernel<<<dim3(nt, nt), dim3(32, 8), 0, h->stream>>>(
            h->ptr<cd>(h->L.S) + (size_t)(2 * i_omega) * strideS, h->ptr<cd>(h->L.S) + (size_t)(2 * i_omega + 1) * strideS,
            h->L.ldS, ng, h->spin_deg / h->vol, (cd *)chi0_out);
    else
        chi0_get_kernel<<<dim3(nt, nt), dim3(32, 8), 0, h->stream>>>(h->ptr<cd>(h->L.S) + (size_t)i_omega * strideS, h->L.ldS, ng,
                                                                     h->spin_deg / h->vol, (cd *)chi0_out);
    h->launches += 1;
    CUDA_TRY(cudaGetLastError());
    return RPA_OK;
}

}  // extern "C"

namespace {
// The blocked Cholesky of the nm matrices of a group (M[0 .. nm), in place; ln det into logdet, flags on a non-positive
// pivot), enqueued on the caller's stream and the handle's side streams: everything between the fork event on the caller's
// stream and the join back onto it.  *launches receives the number of kernels enqueued.
int ec_enqueue_factorization(rpa_chi0 *h, int nm, int n_lanes, int64_t *launches) {
    const Layout &L = h->L;
    const int ng = h->sp.ng;
    cudaStream_t st = h->stream;
    cd *M = h->ptr<cd>(L.M);
    int *d_flag = h->ptr<int>(L.flag);
    double *d_ld = h->ptr<double>(L.logdet);
    const int64_t lt_mat = (int64_t)CH_P * CH_NB * L.ldn;          // per matrix
    const size_t lt_block = (size_t)L.ec_group * lt_mat;           // per block buffer
    const double *wneg = h->ptr<double>(L.wneg);
    struct Lane {
        cudaStream_t main, side;
        cudaEvent_t *ev_panel, ev_col;
        int m0, nm;
    } lanes[EC_MAX_LANES];
    for (int l = 0, m0 = 0; l < n_lanes; l++) {   // matrices dealt as evenly as possible
        const int cnt = nm / n_lanes + (l < nm % n_lanes ? 1 : 0);
        if (l == 0) lanes[l] = {st, h->side, h->ev_panel, h->ev_col, m0, cnt};
        else lanes[l] = {h->xmain[l - 1], h->xside[l - 1], h->xev_panel[l - 1], h->xev_col[l - 1], m0, cnt};
        m0 += cnt;
    }
    auto update = [&](const Lane &ln, cudaStream_t s_, cd *Lt, int K, int g0, int mode, int col_limit) {
        const int rest = ng - g0;
        if (rest <= 0) return 0;
        const int nt = (rest + rk::T - 1) / rk::T;
        const int tiles = mode == 1   ? nt
                          : mode == 2 ? ntiles_lower(rest, rk::T) - nt
                          : mode == 3 ? nt + std::max(nt - 1, 0)
                          : mode == 4 ? (nt > 2 ? (nt - 2) * (nt - 1) / 2 : 0)
                                      : ntiles_lower(rest, rk::T);
        if (tiles <= 0) return 0;
        rank_k_kernel<false><<<dim3(tiles, ln.nm), rk::Cfg<false>::THREADS, rk::Cfg<false>::SMEM_BYTES, s_>>>(
            Lt, L.ldn, lt_mat, K, wneg, CH_P * CH_NB, M + (size_t)ln.m0 * ng * ng, ng, (int64_t)ng * ng, ng, g0, ln.nm, mode,
            col_limit);
        return 1;
    };
    // the updates on the serial chain (strips, look-ahead columns) in 32 x 32 tiles: ncolt column tiles from column g0
    auto update32 = [&](const Lane &ln, cudaStream_t s_, cd *Lt, int K, int g0, int ncolt) {
        const int nt = (ng - g0 + cu32::T - 1) / cu32::T;
        int tiles = 0;
        for (int tj = 0; tj < ncolt; tj++) tiles += std::max(nt - tj, 0);
        if (tiles <= 0) return 0;
        chol_update32_kernel<<<dim3(tiles, ln.nm), cu32::THREADS, cu32::smem_bytes(K), s_>>>(Lt, L.ldn, lt_mat, K,
                                                                                             M + (size_t)ln.m0 * ng * ng, ng, g0, ncolt);
        return 1;
    };
    // which kernel for an update on the chain (ncols64 tile columns of 64 from column g0, all nm matrices of the group):
    // while its 64 x 64 tiles alone fill the GPU the factorisation is throughput-bound and the wide tiles are more
    // efficient (two CTAs per SM, operands through a ring); once they no longer do, the 32 x 32 tiles finish sooner
    auto small_grid = [&](int g0, int ncols64) {
        const int nt = (ng - g0 + rk::T - 1) / rk::T;
        int tiles = 0;
        for (int tj = 0; tj < ncols64; tj++) tiles += std::max(nt - tj, 0);
        return h->ec_tile32 && tiles * nm < 2 * h->n_sm;   // measured on 16 matrices of 401 / 1200 / 3004: 1, 2, 3, 4 x n_sm
    };
    CUDA_TRY(cudaEventRecord(h->ev_fork, st));
    for (int l = 0; l < n_lanes; l++) {
        CUDA_TRY(cudaStreamWaitEvent(lanes[l].side, h->ev_fork, 0));
        if (l > 0) CUDA_TRY(cudaStreamWaitEvent(lanes[l].main, h->ev_fork, 0));
    }
    int blk = 0;
    for (int kb = 0; kb < ng; kb += CH_P * CH_NB, blk++) {
        for (int l = 0; l < n_lanes; l++) {
            const Lane &ln = lanes[l];
            cd *Lt = h->ptr<cd>(L.Lt) + (size_t)(blk & 1) * lt_block + (size_t)ln.m0 * lt_mat;
            // the block's panels and strips: the serial chain, all on the high-priority side stream
            int np = 0;   // panels of this block
            for (int p = 0; p < CH_P && kb + p * CH_NB < ng; p++, np++) {
                const int c0 = kb + p * CH_NB;
                const int rest = ng - (c0 + CH_NB);
                if (p > 0)
                    *launches += small_grid(c0, 1) ? update32(ln, ln.side, Lt, p * CH_NB, c0, 1) : update(ln, ln.side, Lt, p * CH_NB, c0, 1, c0 + CH_NB);
                chol_panel_kernel<<<dim3(std::max(1, (rest + 127) / 128), ln.nm), CH_THREADS, 0, ln.side>>>(
                    M + (size_t)ln.m0 * ng * ng, ng, c0, Lt + (size_t)p * CH_NB * L.ldn, L.ldn, lt_mat, d_flag + ln.m0,
                    d_ld + ln.m0);
                *launches += 1;
            }
            CUDA_TRY(cudaEventRecord(ln.ev_panel[blk & 1], ln.side));
            CUDA_TRY(cudaStreamWaitEvent(ln.main, ln.ev_panel[blk & 1], 0));
            const int g0 = kb + np * CH_NB;
            if (g0 < ng) {
                // look-ahead: the first two tile columns (= the next block's 128 columns) on the side stream, after
                // the previous block's big update; the rest of the trailing matrix on the main stream meanwhile
                if (blk > 0) CUDA_TRY(cudaStreamWaitEvent(ln.side, ln.ev_col, 0));
                *launches += small_grid(g0, 2) ? update32(ln, ln.side, Lt, np * CH_NB, g0, 2 * rk::T / cu32::T) : update(ln, ln.side, Lt, np * CH_NB, g0, 3, ng);
                *launches += update(ln, ln.main, Lt, np * CH_NB, g0, 4, ng);
                CUDA_TRY(cudaEventRecord(ln.ev_col, ln.main));
            }
        }
    }
    for (int l = 1; l < n_lanes; l++) {   // join: the caller's stream continues after the other lanes
        CUDA_TRY(cudaEventRecord(h->xev_join[l - 1], lanes[l].main));
        CUDA_TRY(cudaStreamWaitEvent(st, h->xev_join[l - 1], 0));
    }
    CUDA_TRY(cudaGetLastError());
    return RPA_OK;
}

// The same through a CUDA graph: the factorisation of a group is ~170 (1 lane) to ~600 (4 lanes) small dependent launches
// on up to eight streams, and issuing them costs the host more than the device needs to run them (every lane adds its own
// launches and event operations to the one issuing thread).  The launch sequence depends only on (nm, n_lanes) -- all
// pointers lie in the caller's workspace -- so it is captured once per handle and shape and replayed with one
// cudaGraphLaunch.  Falls back to direct launches if capture or instantiation fails.
int ec_factorize(rpa_chi0 *h, int nm, int n_lanes) {
    if (h->ec_use_graph) {
        for (auto &g : h->ec_graphs)
            if (g.nm == nm && g.lanes == n_lanes) {
                CUDA_TRY(cudaGraphLaunch(g.exec, h->stream));
                h->launches += g.launches;
                return RPA_OK;
            }
        if (h->ec_graphs.size() < 16) {
            int64_t n = 0;
            cudaGraph_t graph = nullptr;
            cudaGraphExec_t exec = nullptr;
            bool ok = cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
            if (ok) {
                const int rc = ec_enqueue_factorization(h, nm, n_lanes, &n);
                const cudaError_t e = cudaStreamEndCapture(h->stream, &graph);
                ok = rc == RPA_OK && e == cudaSuccess && graph != nullptr;
            }
            if (ok) ok = cudaGraphInstantiate(&exec, graph, 0) == cudaSuccess;
            if (graph) cudaGraphDestroy(graph);
            if (ok) {
                h->ec_graphs.push_back({nm, n_lanes, exec, n});
                CUDA_TRY(cudaGraphLaunch(exec, h->stream));
                h->launches += n;
                return RPA_OK;
            }
            cudaGetLastError();          // clear the capture error
            h->ec_use_graph = false;     // and stay on direct launches
        }
    }
    int64_t n = 0;
    const int rc = ec_enqueue_factorization(h, nm, n_lanes, &n);
    h->launches += n;
    return rc;
}

// e(omega_i) for i in [iw_begin, iw_end) and ec = (1/2pi) sum over that range of wt_i e_i
int ec_q_impl(rpa_chi0_t *h, const double *v_G, int iw_begin, int iw_end, double *ec_ha, double *e_omega) {
    if (!h || !v_G || !ec_ha) return fail(RPA_ERR_INVALID_ARG, "rpa_ec_q: NULL argument");
    if (h->eta > 0.0) return fail(RPA_ERR_UNSUPPORTED, "rpa_ec_q: Eq. 2 is an imaginary-axis integral; this is a real-axis handle");
    if (!h->has_wt) return fail(RPA_ERR_INVALID_ARG, "rpa_ec_q: omega_wt was NULL at create");
    if (iw_begin < 0 || iw_end > h->n_omega || iw_begin > iw_end)
        return fail(RPA_ERR_INVALID_ARG, "rpa_ec_q_range: frequency range [%d, %d) outside [0, %d)", iw_begin, iw_end, h->n_omega);
    const Layout &L = h->L;
    const int ng = h->sp.ng;
    for (int i = 0; i < ng; i++)
        if (!(v_G[i] > 0.0) || !std::isfinite(v_G[i])) return fail(RPA_ERR_INVALID_ARG, "rpa_ec_q: v_G[%d] must be finite and > 0", i);
    cudaStream_t st = h->stream;
    double *d_v = h->ptr<double>(L.v), *d_e = h->ptr<double>(L.e), *d_tr = h->ptr<double>(L.tr), *d_ld = h->ptr<double>(L.logdet);
    int *d_flag = h->ptr<int>(L.flag);
    cd *M = h->ptr<cd>(L.M);
    const cd *S = h->ptr<cd>(L.S);
    const int64_t strideS = (int64_t)ng * L.ldS;
    const double scale = h->spin_deg / h->vol;
    CUDA_TRY(cudaMemcpyAsync(d_v, v_G, ng * sizeof(double), cudaMemcpyHostToDevice, st));
    for (int iw0 = iw_begin; iw0 < iw_end; iw0 += L.ec_group) {
        const int nm = std::min(L.ec_group, iw_end - iw0);
        CUDA_TRY(cudaMemsetAsync(d_ld, 0, EC_GROUP * sizeof(double), st));
        CUDA_TRY(cudaMemsetAsync(d_flag, 0, EC_GROUP * sizeof(int), st));
        ec_build_kernel<<<dim3((ng + 127) / 128, ng, nm), 128, 0, st>>>(S + (size_t)iw0 * strideS, L.ldS, strideS, ng, scale, d_v, M);
        ec_trace_kernel<<<nm, 256, 0, st>>>(S + (size_t)iw0 * strideS, L.ldS, strideS, ng, scale, d_v, d_tr);
        h->launches += 2;
        // Blocked right-looking Cholesky, left-looking inside a block of CH_P panels (CH_P * 32 = 128 columns): panel p of
        // a block first receives the updates of the block's earlier panels on its own 32 columns (a strip: first tile
        // column of rank_k_kernel<false>, K = 32 p, columns limited to the panel), is factored and solved, and only after
        // the last panel is the trailing matrix updated, once, with K = 128: the read-modify-write of the trailing matrix
        // (0.37 GB for cfg 1, beyond L2) happens once per 128 columns instead of once per 32.
        // Look-ahead: the next block needs only the first two tile columns (128 columns) of that big update; they are
        // updated on the high-priority side stream, which then runs the whole next block (panels and strips: the serial,
        // latency-bound chain) while the rest of the update proceeds on the main stream.  Two block buffers of Lt alternate
        // (block b + 2 starts after the look-ahead of block b + 1, which waits for the big update of block b).
        // Lanes: the group's matrices are split in shares that run the same schedule on their own pair of streams.
        // The panel steps are latency-bound (one warp factors the diagonal block, few CTAs), the trailing updates are
        // throughput-bound: with independent shares in flight one share's updates fill the SMs while another is in
        // its panel steps.  Two lanes by default; rpa_chi0_set_ec_lanes(h, n) (1 ... 4) chooses (measured on 16 matrices of 1200
        // with the whole-block look-ahead: 2.68 / 2.66 / 2.64 / 2.63 ms for 1 / 2 / 3 / 4 lanes: the chain of a lane
        // does not get shorter, so more lanes add little).
        const int n_lanes = std::max(1, std::min({h->ec_lanes, EC_MAX_LANES, nm}));
        {
            const int rc = ec_factorize(h, nm, n_lanes);
            if (rc != RPA_OK) return rc;
        }
        CUDA_TRY(cudaGetLastError());
        ec_collect_kernel<<<1, 32, 0, st>>>(d_ld, d_tr, nm, iw0, d_e);
        h->launches += 1;
        int flags[EC_GROUP] = {0, 0, 0, 0};
        CUDA_TRY(cudaMemcpyAsync(flags, d_flag, EC_GROUP * sizeof(int), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
        for (int i = 0; i < nm; i++)
            if (flags[i]) return fail(RPA_ERR_NOT_PD, "rpa_ec_q: I - v^1/2 chi0 v^1/2 not positive definite at omega index %d", iw0 + i);
    }
    ec_sum_kernel<<<1, 32, 0, st>>>(d_e + iw_begin, h->ptr<double>(L.wt) + iw_begin, iw_end - iw_begin, h->ptr<double>(L.ec));
    h->launches += 1;
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaMemcpyAsync(ec_ha, h->ptr<double>(L.ec), sizeof(double), cudaMemcpyDeviceToHost, st));
    if (e_omega && iw_end > iw_begin)
        CUDA_TRY(cudaMemcpyAsync(e_omega, d_e + iw_begin, (iw_end - iw_begin) * sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return RPA_OK;
}
}  // namespace

extern "C" {

int rpa_ec_q(rpa_chi0_t *h, const double *v_G, double *ec_ha, double *e_omega) {
    return ec_q_impl(h, v_G, 0, h ? h->n_omega : 0, ec_ha, e_omega);
}

int rpa_ec_q_range(rpa_chi0_t *h, const double *v_G, int32_t iw_begin, int32_t iw_end, double *ec_partial_ha, double *e_omega) {
    return ec_q_impl(h, v_G, iw_begin, iw_end, ec_partial_ha, e_omega);
}

int rpa_chi0_reset(rpa_chi0_t *h) {
    if (!h) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_reset: handle is NULL");
    CUDA_TRY(cudaMemsetAsync(h->ws + h->L.S, 0, (size_t)h->n_omega * h->sp.ng * h->L.ldS * sizeof(cd), h->stream));
    return RPA_OK;
}

int rpa_chi0_set_spin_degeneracy(rpa_chi0_t *h, int32_t s) {
    if (!h) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_set_spin_degeneracy: handle is NULL");
    if (s != 1 && s != 2) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_set_spin_degeneracy: s must be 1 or 2, got %d", s);
    h->spin_deg = (double)s;
    return RPA_OK;
}

int rpa_chi0_set_rank_k_mode(rpa_chi0_t *h, int32_t mode, int32_t digits) {
    if (!h) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_set_rank_k_mode: handle is NULL");
    const int kind = mode & 0xff, flags = mode & ~0xff;
    if (flags & ~(RPA_RANK_K_FLAG_NO_CLUSTER | RPA_RANK_K_FLAG_ALL_BATCHES))
        return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_set_rank_k_mode: unknown flag bits 0x%x", flags);
    if (kind == RPA_RANK_K_FP64_3M || kind == RPA_RANK_K_FP64_4M) {
        if (flags) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_set_rank_k_mode: flags apply to RPA_RANK_K_I8 only");
        h->use_i8 = false;
        h->use_3m = kind == RPA_RANK_K_FP64_3M;
        return RPA_OK;
    }
    if (kind != RPA_RANK_K_I8) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_set_rank_k_mode: unknown mode %d", kind);
    if (digits == 0) digits = 7;
    if (digits < 6 || digits > 8) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_set_rank_k_mode: digits must be 6, 7 or 8 (0: 7), got %d", digits);
    if (!h->i8_attr_set) {
        CUDA_TRY(cudaFuncSetAttribute(rank_k_i8_kernel<6, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, rki8::smem_bytes(6)));
        CUDA_TRY(cudaFuncSetAttribute(rank_k_i8_kernel<7, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, rki8::smem_bytes(7)));
        CUDA_TRY(cudaFuncSetAttribute(rank_k_i8_kernel<8, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, rki8::smem_bytes(8)));
        CUDA_TRY(cudaFuncSetAttribute(rank_k_i8_kernel<6, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, rki8::smem_bytes(6)));
        CUDA_TRY(cudaFuncSetAttribute(rank_k_i8_kernel<7, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, rki8::smem_bytes(7)));
        CUDA_TRY(cudaFuncSetAttribute(rank_k_i8_kernel<8, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, rki8::smem_bytes(8)));
        h->i8_attr_set = true;
    }
    h->i8_cluster = !(flags & RPA_RANK_K_FLAG_NO_CLUSTER);
    h->i8_force = (flags & RPA_RANK_K_FLAG_ALL_BATCHES) != 0;
    h->i8_digits = digits;
    h->use_3m = true;   // batches the int8 path does not take run rank_k3m_kernel
    // tiles (128-row block of L, 64-column block) that meet the lower triangle of either half (Re, Im) of D = L R^T
    h->i8_tiles.clear();
    const int ng_ = h->sp.ng, ngp = (ng_ + rki8::RB - 1) / rki8::RB * rki8::RB;
    for (int rb = 0; rb < 2 * ngp / rki8::RB; rb++) {
        const int g_lo = (rb * rki8::RB) % ngp, g_hi = std::min(g_lo + rki8::RB - 1, ng_ - 1);
        if (g_lo >= ng_) continue;
        int cb = 0;
        for (; cb * rki8::CB <= g_hi; cb++) h->i8_tiles.push_back(make_int2(rb, cb));
        // clusters of two CTAs share a row block: an odd row gets a padding tile beyond the triangle (stores nothing)
        if (h->i8_cluster && (cb & 1)) h->i8_tiles.push_back(make_int2(rb, cb));
    }
    h->use_i8 = true;
    return RPA_OK;
}

int rpa_chi0_rank_k_batches(const rpa_chi0_t *h, int64_t *fp64_batches, int64_t *i8_batches) {
    if (!h || !fp64_batches || !i8_batches) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_rank_k_batches: NULL argument");
    *fp64_batches = h->fp64_batches;
    *i8_batches = h->i8_batches;
    return RPA_OK;
}

int rpa_chi0_set_ec_lanes(rpa_chi0_t *h, int32_t n_lanes) {
    if (!h) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_set_ec_lanes: handle is NULL");
    const bool wide = (n_lanes & RPA_EC_FLAG_WIDE_TILES) != 0;
    n_lanes &= ~RPA_EC_FLAG_WIDE_TILES;
    if (n_lanes < 1 || n_lanes > EC_MAX_LANES)
        return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_set_ec_lanes: n_lanes must be 1 ... %d, got %d", EC_MAX_LANES, n_lanes);
    if (h->ec_tile32 == wide) {   // the captured graphs hold the other kernels
        for (auto &g : h->ec_graphs) cudaGraphExecDestroy(g.exec);
        h->ec_graphs.clear();
    }
    h->ec_tile32 = !wide;
    h->ec_lanes = n_lanes;
    return RPA_OK;
}

// E_c = sum_q w_q E_c(q): the outer q loop's final sum of Eq. 1 over the IBZ weights.  Host arithmetic on the
// per-q scalars rpa_ec_q returned; summed in the order given.
int rpa_total_energy(int32_t n_q, const double *ec_q, const double *q_weights, double *ec_ha) {
    if (n_q < 0 || !ec_ha || (n_q > 0 && (!ec_q || !q_weights))) return fail(RPA_ERR_INVALID_ARG, "rpa_total_energy: invalid argument");
    double sum = 0.0;
    for (int i = 0; i < n_q; i++) sum += q_weights[i] * ec_q[i];
    *ec_ha = sum;
    return RPA_OK;
}

int rpa_chi0_sync(rpa_chi0_t *h) {
    if (!h) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_sync: handle is NULL");
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    CUDA_TRY(cudaGetLastError());
    return RPA_OK;
}

int rpa_chi0_set_profiling(rpa_chi0_t *h, int32_t on) {
    if (!h) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_set_profiling: handle is NULL");
    int rc = drain_events(h);
    if (rc != RPA_OK) return rc;
    h->prof = on != 0;
    for (int i = 0; i < NSTAGE; i++) { h->stage_ms[i] = 0.0; h->stage_launches[i] = 0; }
    return RPA_OK;
}

int rpa_chi0_stage_times(rpa_chi0_t *h, double ms[6], int64_t launches[6]) {
    if (!h || !ms || !launches) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_stage_times: NULL argument");
    int rc = drain_events(h);
    if (rc != RPA_OK) return rc;
    for (int i = 0; i < NSTAGE; i++) { ms[i] = h->stage_ms[i]; launches[i] = h->stage_launches[i]; }
    return RPA_OK;
}

int rpa_chi0_launch_count(const rpa_chi0_t *h, int64_t *count) {
    if (!h || !count) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_launch_count: NULL argument");
    *count = h->launches;
    return RPA_OK;
}

int rpa_chi0_accumulators(const rpa_chi0_t *h, void **S, size_t *bytes) {
    if (!h || !S || !bytes) return fail(RPA_ERR_INVALID_ARG, "rpa_chi0_accumulators: NULL argument");
    *S = h->ws + h->L.S;
    *bytes = (size_t)h->n_omega * h->sp.ng * h->L.ldS * sizeof(cd);
    return RPA_OK;
}

void rpa_chi0_destroy(rpa_chi0_t *h) {
    if (!h) return;
    if (h->side) cudaStreamDestroy(h->side);
    for (cudaEvent_t e : {h->ev_panel[0], h->ev_panel[1], h->ev_col, h->ev_fork})
        if (e) cudaEventDestroy(e);
    for (int l = 0; l < EC_MAX_LANES - 1; l++) {
        for (cudaStream_t s_ : {h->xside[l], h->xmain[l]})
            if (s_) cudaStreamDestroy(s_);
        for (cudaEvent_t e : {h->xev_panel[l][0], h->xev_panel[l][1], h->xev_col[l], h->xev_join[l]})
            if (e) cudaEventDestroy(e);
    }
    for (auto &g : h->ec_graphs) cudaGraphExecDestroy(g.exec);
    for (auto &ev : h->events) { cudaEventDestroy(ev.a); cudaEventDestroy(ev.b); }
    for (auto &e : h->pool) cudaEventDestroy(e);
    delete h;
}

// ---- Table 1 steps 3-4: plane-wave coefficients -> grid orbitals (Eq. 10), IBZ -> BZ remap (Eq. 11) -----------------
int rpa_pw_to_grid(rpa_chi0_t *h, int32_t n_bands, int32_t n_pw, const int32_t *g_pw, const void *C, void *psi_out) {
    if (!h) return fail(RPA_ERR_INVALID_ARG, "rpa_pw_to_grid: handle is NULL");
    if (n_bands < 0 || n_pw < 0) return fail(RPA_ERR_INVALID_ARG, "rpa_pw_to_grid: negative count");
    if (n_bands == 0) return RPA_OK;
    if (!psi_out || (n_pw > 0 && (!g_pw || !C))) return fail(RPA_ERR_INVALID_ARG, "rpa_pw_to_grid: NULL array");
    const Layout &L = h->L;
    cudaStream_t st = h->stream;
    const int N1 = h->grid[0], N2 = h->grid[1], N3 = h->grid[2];
    const size_t N = (size_t)N1 * N2 * N3;
    if (n_pw == 0) {
        CUDA_TRY(cudaMemsetAsync(psi_out, 0, (size_t)n_bands * N * sizeof(cd), st));
        return RPA_OK;
    }
    // The table box index -> coefficient index depends only on g_pw: callers expand many band sets with the same vectors
    // (every k-point slice, every step), so the last table stays on the device in its own workspace region and a call
    // with the same g_pw neither rebuilds nor uploads it (and does not wait for the stream).
    const bool cached = h->pw_g.size() == (size_t)3 * n_pw && memcmp(h->pw_g.data(), g_pw, (size_t)3 * n_pw * sizeof(int32_t)) == 0;
    int qmin[3], qmax[3];
    int64_t nq1, nq2, nq3;
    if (cached) {
        for (int d = 0; d < 3; d++) qmin[d] = h->pw_qmin[d];
        nq1 = h->pw_nq[0]; nq2 = h->pw_nq[1]; nq3 = h->pw_nq[2];
    } else {
        for (int d = 0; d < 3; d++) qmin[d] = qmax[d] = g_pw[d];
        for (int i = 0; i < n_pw; i++)
            for (int d = 0; d < 3; d++) {
                qmin[d] = std::min(qmin[d], (int)g_pw[3 * i + d]);
                qmax[d] = std::max(qmax[d], (int)g_pw[3 * i + d]);
            }
        nq1 = (int64_t)qmax[0] - qmin[0] + 1; nq2 = (int64_t)qmax[1] - qmin[1] + 1; nq3 = (int64_t)qmax[2] - qmin[2] + 1;
    }
    const int64_t ncol = nq2 * nq3;
    const size_t scratch = (size_t)L.sub_pairs * L.I_pair_bytes;
    const bool keep = nq1 * ncol <= (int64_t)N;   // fits the table region (a box inside the grid always does)
    const size_t table_bytes = keep ? 0 : align_up((size_t)(nq1 * ncol) * sizeof(int32_t), 256);
    const size_t t1_band = (size_t)N1 * ncol * sizeof(cd);
    const size_t smem = ((size_t)N2 + N3 + ncol + (size_t)N2 * nq3) * sizeof(cd);
    if (nq1 * ncol > ((int64_t)1 << 28) || table_bytes + t1_band > scratch)
        return fail(RPA_ERR_WORKSPACE, "rpa_pw_to_grid: plane-wave box %lld x %lld x %lld does not fit the handle's scratch (%zu B)",
                    (long long)nq1, (long long)nq2, (long long)nq3, scratch);
    if (smem > 200 * 1024)
        return fail(RPA_ERR_UNSUPPORTED, "rpa_pw_to_grid: plane of the plane-wave box too large for shared memory (%zu B)", smem);
    unsigned char *base = h->ws + L.I;
    int32_t *d_table = keep ? h->ptr<int32_t>(L.pwtab) : reinterpret_cast<int32_t *>(base);
    cd *T1 = reinterpret_cast<cd *>(base + table_bytes);
    if (!cached) {
        h->pw_g.clear();   // no table is valid while this one is being built
        std::vector<int32_t> &table = h->pw_table;
        table.assign((size_t)(nq1 * ncol), -1);
        for (int i = 0; i < n_pw; i++) {
            const size_t at = ((size_t)(g_pw[3 * i] - qmin[0]) * nq2 + (g_pw[3 * i + 1] - qmin[1])) * nq3 + (g_pw[3 * i + 2] - qmin[2]);
            if (table[at] >= 0) return fail(RPA_ERR_INVALID_ARG, "rpa_pw_to_grid: plane wave %d duplicates plane wave %d", i, table[at]);
            table[at] = i;
        }
        CUDA_TRY(cudaMemcpyAsync(d_table, table.data(), table.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
        CUDA_TRY(cudaStreamSynchronize(st));   // `table` is pageable host memory that the next call may rewrite
        if (keep) {
            h->pw_g.assign(g_pw, g_pw + (size_t)3 * n_pw);
            for (int d = 0; d < 3; d++) h->pw_qmin[d] = qmin[d];
            h->pw_nq[0] = nq1; h->pw_nq[1] = nq2; h->pw_nq[2] = nq3;
        }
    }
    const PwZyKernel zy = pw_zy_pick(N2, N3);
    if (smem > 48 * 1024) CUDA_TRY(cudaFuncSetAttribute(zy, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    // table-driven persistent kernel when both in-plane axes have a radix-8 / radix-12 split and its arrays fit
    PwZyTabKernel zy_tab = pw_zy_tab_pick(N2, N3);
    PwTabDims td{};
    int tab_ctas = 0;
    if (zy_tab) {
        td = pw_tab_dims(N2, N3, pw_pick_na(N2), pw_pick_na(N3), qmin[1], (int)nq2, qmin[2], (int)nq3);
        if (td.smem > 200 * 1024) {
            zy_tab = nullptr;
        } else {
            if (td.smem > 48 * 1024)
                CUDA_TRY(cudaFuncSetAttribute(zy_tab, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)td.smem));
            CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&tab_ctas, zy_tab, 128, td.smem));
            if (tab_ctas < 1) zy_tab = nullptr;
        }
    }
    const int chunk = (int)std::min<size_t>((size_t)n_bands, std::min<size_t>(65535, (scratch - table_bytes) / t1_band));
    for (int b0 = 0; b0 < n_bands; b0 += chunk) {
        const int nb = std::min(chunk, n_bands - b0);
        const int na1 = pw_pick_na(N1);
        pw_xaxis_pick(na1)<<<dim3((unsigned)((ncol + 127) / 128), N1 / na1, nb), 128, 0, st>>>(
            (const cd *)C + (size_t)b0 * n_pw, n_pw, d_table, h->ptr<cd>(L.tw1), N1, qmin[0], (int)nq1, (int)ncol, T1);
        if (zy_tab) {
            const int n_items = nb * N1;
            zy_tab<<<std::min(n_items, h->n_sm * tab_ctas), 128, td.smem, st>>>(
                T1, h->ptr<cd>(L.tw2), h->ptr<cd>(L.tw3), N1, N2, N3, qmin[1], (int)nq2, qmin[2], (int)nq3, n_items,
                (cd *)psi_out + (size_t)b0 * N);
        } else {
            zy<<<dim3(N1, nb), 128, smem, st>>>(T1, h->ptr<cd>(L.tw2), h->ptr<cd>(L.tw3), N1, N2, N3, qmin[1], (int)nq2, qmin[2],
                                               (int)nq3, (cd *)psi_out + (size_t)b0 * N);
        }
        h->launches += 2;
        CUDA_TRY(cudaGetLastError());
    }
    return RPA_OK;
}

int rpa_symmetry_remap(rpa_chi0_t *h, int32_t n_bands, const int32_t M[9], int32_t time_reversal, const void *psi_in,
                       void *psi_out) {
    if (!h || !M) return fail(RPA_ERR_INVALID_ARG, "rpa_symmetry_remap: NULL argument");
    if (n_bands < 0) return fail(RPA_ERR_INVALID_ARG, "rpa_symmetry_remap: negative count");
    if (n_bands == 0) return RPA_OK;
    if (!psi_in || !psi_out || psi_in == psi_out) return fail(RPA_ERR_INVALID_ARG, "rpa_symmetry_remap: NULL or aliased arrays");
    RemapParams R;
    R.N1 = h->grid[0]; R.N2 = h->grid[1]; R.N3 = h->grid[2];
    R.conj = time_reversal != 0;
    for (int i = 0; i < 3; i++)
        for (int k = 0; k < 3; k++) {
            const int64_t num = (int64_t)M[3 * i + k] * h->grid[i];
            if (num % h->grid[k] != 0)
                return fail(RPA_ERR_UNSUPPORTED, "rpa_symmetry_remap: the operation does not map the grid onto itself (M[%d][%d])", i, k);
            R.S[3 * i + k] = (int)(num / h->grid[k]);
        }
    const int64_t N = (int64_t)R.N1 * R.N2 * R.N3;
    for (int b0 = 0; b0 < n_bands; b0 += 65535) {
        const int nb = std::min(65535, n_bands - b0);
        symmetry_remap_kernel<<<dim3((unsigned)((N + 255) / 256), nb), 256, 0, h->stream>>>(
            (const cd *)psi_in + (size_t)b0 * N, (cd *)psi_out + (size_t)b0 * N, R);
        h->launches += 1;
    }
    CUDA_TRY(cudaGetLastError());
    return RPA_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// rpa_e_omega_noalloc: e(omega) of Eq. 2 for one caller-supplied chi0 matrix, without any device allocation
// (include/rpa_chi0.h).  The matrix being factorised, the solved panels of a block and the scalars live in ONE
// file-scope device array; every GPU that loads the library holds it until the process exits.
//
// In host code `rpa_noalloc_scratch` is a host-side stand-in for the symbol, not a device address: the address the
// kernels get is the one cudaGetSymbolAddress returns, taken once per device with that device current (noalloc_setup).
namespace {
constexpr int NA_MAX_NG = RPA_NOALLOC_MAX_NG;
constexpr size_t NA_M = 0;                                                    // cd [ng][ng]: 1 - v^1/2 chi0 v^1/2, factorised in place
constexpr size_t NA_LT = NA_M + (size_t)NA_MAX_NG * NA_MAX_NG * sizeof(cd);   // cd [CH_P * CH_NB][ldn]: solved panels of the current block
constexpr size_t NA_WNEG = NA_LT + (size_t)CH_P * CH_NB * NA_MAX_NG * sizeof(cd);   // double [CH_P * CH_NB] = -1: weight of the trailing update
constexpr size_t NA_LOGDET = NA_WNEG + (size_t)CH_P * CH_NB * sizeof(double);
constexpr size_t NA_TR = NA_LOGDET + 256;
constexpr size_t NA_FLAG = NA_TR + 256;
constexpr size_t NA_BYTES = NA_FLAG + 512;
static_assert(NA_BYTES == RPA_NOALLOC_SCRATCH_BYTES, "the header states the size of the array");
static_assert(NA_LT % 256 == 0 && NA_WNEG % 256 == 0 && NA_LOGDET % 256 == 0, "sub-buffers stay 256-byte aligned");
constexpr int NA_MAX_DEVICES = 64;
}  // namespace

static __device__ __align__(256) unsigned char rpa_noalloc_scratch[NA_BYTES];

// what every call must find initialised, whatever the last call left: the update weights, ln det = 0, flag = 0
__global__ void noalloc_begin_kernel(double *__restrict__ wneg, double *__restrict__ logdet, int *__restrict__ flag) {
    const int i = threadIdx.x;
    if (i < CH_P * CH_NB) wneg[i] = -1.0;
    if (i == 0) {
        *logdet = 0.0;
        *flag = 0;
    }
}

// e = ln det + Tr, NaN after a non-positive pivot
__global__ void noalloc_finish_kernel(const double *__restrict__ logdet, const double *__restrict__ tr,
                                      const int *__restrict__ flag, double *__restrict__ e) {
    if (threadIdx.x == 0) *e = *flag ? __longlong_as_double(0x7ff8000000000000ll) : *logdet + *tr;
}

namespace {
struct NoallocDevice {
    bool ready = false;
    unsigned char *scratch = nullptr;   // DEVICE address of rpa_noalloc_scratch on this device
};
NoallocDevice g_noalloc[NA_MAX_DEVICES];
std::mutex g_noalloc_mutex;

// once per device, with that device current: the device address of the array, and the shared-memory size of the update kernel
int noalloc_setup(int dev, unsigned char **scratch) {
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    NoallocDevice &d = g_noalloc[dev];
    if (!d.ready) {
        unsigned char *p = nullptr;
        CUDA_TRY(cudaGetSymbolAddress((void **)&p, rpa_noalloc_scratch));
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255) != 0)
            return fail(RPA_ERR_CUDA, "rpa_e_omega_noalloc: cudaGetSymbolAddress gave %p for the scratch array", (void *)p);
        CUDA_TRY(cudaFuncSetAttribute(rank_k_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, rk::Cfg<false>::SMEM_BYTES));
        d.scratch = p;
        d.ready = true;
    }
    *scratch = d.scratch;
    return RPA_OK;
}
}  // namespace

extern "C" int rpa_e_omega_noalloc(const void *chi0, int32_t ng, const double *v_G, double *e, void *cuda_stream) {
    if (!chi0 || !v_G || !e) return fail(RPA_ERR_INVALID_ARG, "rpa_e_omega_noalloc: NULL argument");
    if (ng < 1) return fail(RPA_ERR_INVALID_ARG, "rpa_e_omega_noalloc: ng = %d", ng);
    if (ng > NA_MAX_NG)
        return fail(RPA_ERR_UNSUPPORTED, "rpa_e_omega_noalloc: ng = %d exceeds RPA_NOALLOC_MAX_NG = %d (the fixed scratch array); use rpa_ec_q",
                    ng, NA_MAX_NG);
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NA_MAX_DEVICES) return fail(RPA_ERR_UNSUPPORTED, "rpa_e_omega_noalloc: device ordinal %d", dev);
    unsigned char *scratch = nullptr;
    {
        const int rc = noalloc_setup(dev, &scratch);
        if (rc != RPA_OK) return rc;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cd *M = reinterpret_cast<cd *>(scratch + NA_M), *Lt = reinterpret_cast<cd *>(scratch + NA_LT);
    double *wneg = reinterpret_cast<double *>(scratch + NA_WNEG), *logdet = reinterpret_cast<double *>(scratch + NA_LOGDET);
    double *tr = reinterpret_cast<double *>(scratch + NA_TR);
    int *flag = reinterpret_cast<int *>(scratch + NA_FLAG);
    const cd *X = static_cast<const cd *>(chi0);
    const int64_t ldn = (int64_t)align_up((size_t)ng, 8);
    const int64_t lt_mat = (int64_t)CH_P * CH_NB * ldn;

    noalloc_begin_kernel<<<1, CH_P * CH_NB, 0, st>>>(wneg, logdet, flag);
    // chi0 is already (s / Omega) S: scale 1
    ec_build_kernel<<<dim3((ng + 127) / 128, ng, 1), 128, 0, st>>>(X, ng, 0, ng, 1.0, v_G, M);
    ec_trace_kernel<<<1, 256, 0, st>>>(X, ng, 0, ng, 1.0, v_G, tr);
    // the schedule of rpa_ec_q for one matrix on one stream: per block of CH_P panels, panel p first receives the
    // block's earlier panels on its own 32 columns (strip), is factored and solved; then one K = 128 trailing update
    auto update = [&](int K, int g0, int mode, int col_limit) {
        const int rest = ng - g0;
        if (rest <= 0) return;
        const int nt = (rest + rk::T - 1) / rk::T;
        const int tiles = mode == 1 ? nt : ntiles_lower(rest, rk::T);
        rank_k_kernel<false><<<dim3(tiles, 1), rk::Cfg<false>::THREADS, rk::Cfg<false>::SMEM_BYTES, st>>>(
            Lt, ldn, lt_mat, K, wneg, CH_P * CH_NB, M, ng, (int64_t)ng * ng, ng, g0, 1, mode, col_limit);
    };
    for (int kb = 0; kb < ng; kb += CH_P * CH_NB) {
        int np = 0;
        for (int p = 0; p < CH_P && kb + p * CH_NB < ng; p++, np++) {
            const int c0 = kb + p * CH_NB;
            const int rest = ng - (c0 + CH_NB);
            if (p > 0) update(p * CH_NB, c0, 1, c0 + CH_NB);
            chol_panel_kernel<<<dim3(std::max(1, (rest + 127) / 128), 1), CH_THREADS, 0, st>>>(
                M, ng, c0, Lt + (size_t)p * CH_NB * ldn, ldn, lt_mat, flag, logdet);
        }
        update(np * CH_NB, kb + np * CH_NB, 0, ng);
    }
    noalloc_finish_kernel<<<1, 32, 0, st>>>(logdet, tr, flag, e);
    CUDA_TRY(cudaGetLastError());
    return RPA_OK;
}
