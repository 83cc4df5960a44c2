// PAW one-centre correction (Eq. 6; Table 1 steps 8-9):
//   n_nm(g) = ntilde_nm(g) + sum_a exp(-i K_g . R_a) sum_ij conj(P^a_i,n) Q^a_ij(g) P^a_j,m .
// Re-associated so that everything depending on the occupied band n alone is done once per n:
//   T_n[a,j][g] = exp(-i K_g . R_a) sum_i conj(P^a_i,n) Q^a_ij(g)          (paw_T_kernel)
//   n_nm(g)    += sum_{a,j} P^a_j,m T_n[a,j][g]                             (paw_add_kernel, a small complex GEMM)
// which is the same sum in a different order (8 sum_a n_a nG flop per pair instead of 8 sum_a n_a^2 nG).
// Ragged atoms (different projector counts) are handled through the per-projector index arrays.
#pragma once
#include "common.cuh"

// grid (ceil(ng/128), ptot, nslots); T[(slot*ptot + aj)*ldn + g]
__global__ void __launch_bounds__(128)
paw_T_kernel(cd *__restrict__ T, int64_t ldn, int ng, int ptot, const cd *__restrict__ P_occ, int n0,
             const cd *__restrict__ Q, const int32_t *__restrict__ aj_atom, const int32_t *__restrict__ aj_j,
             const int32_t *__restrict__ atom_poff, const int32_t *__restrict__ atom_ni,
             const int64_t *__restrict__ atom_qoff, const double *__restrict__ R, const double *__restrict__ Kc) {
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= ng) return;
    const int aj = blockIdx.y, slot = blockIdx.z;
    const int a = aj_atom[aj], j = aj_j[aj];
    const int ni = atom_ni[a], poff = atom_poff[a];
    const cd *Pn = P_occ + (size_t)(n0 + slot) * ptot + poff;
    const cd *Qa = Q + atom_qoff[a] + (size_t)j * ng + g;
    cd acc = cmake(0.0, 0.0);
    for (int i = 0; i < ni; i++) {
        const cd p = Pn[i];
        const cd q = Qa[(size_t)i * ni * ng];
        acc = cfma(cmake(p.x, -p.y), q, acc);
    }
    const double kr = Kc[3 * g] * R[3 * a] + Kc[3 * g + 1] * R[3 * a + 1] + Kc[3 * g + 2] * R[3 * a + 2];
    double sn, cs;
    sincos(kr, &sn, &cs);
    T[((size_t)slot * ptot + aj) * ldn + g] = cmul(cmake(cs, -sn), acc);
}

// grid (ceil(ng/128), nslots * ceil(mlen/PAW_PB)); pair p = slot*mlen + mm.
#define PAW_PB 8
#define PAW_AJ_TILE 64
__global__ void __launch_bounds__(128)
paw_add_kernel(cd *__restrict__ Nbuf, int64_t ldn, int ng, int ptot, const cd *__restrict__ T,
               const cd *__restrict__ P_unocc, int mlen, int m0) {
    __shared__ cd Ps[PAW_PB][PAW_AJ_TILE];
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    const int chunks = (mlen + PAW_PB - 1) / PAW_PB;
    const int slot = blockIdx.y / chunks, mm0 = (blockIdx.y % chunks) * PAW_PB;
    const int np = min(PAW_PB, mlen - mm0);
    cd acc[PAW_PB];
#pragma unroll
    for (int u = 0; u < PAW_PB; u++) acc[u] = cmake(0.0, 0.0);
    const cd *Ts = T + (size_t)slot * ptot * ldn;
    for (int aj0 = 0; aj0 < ptot; aj0 += PAW_AJ_TILE) {
        const int na = min(PAW_AJ_TILE, ptot - aj0);
        __syncthreads();
        for (int i = threadIdx.x; i < PAW_PB * PAW_AJ_TILE; i += blockDim.x) {
            const int u = i / PAW_AJ_TILE, k = i % PAW_AJ_TILE;
            Ps[u][k] = (u < np && k < na) ? P_unocc[(size_t)(m0 + mm0 + u) * ptot + aj0 + k] : cmake(0.0, 0.0);
        }
        __syncthreads();
        if (g < ng) {
            for (int k = 0; k < na; k++) {
                const cd tv = Ts[(size_t)(aj0 + k) * ldn + g];
#pragma unroll
                for (int u = 0; u < PAW_PB; u++) acc[u] = cfma(Ps[u][k], tv, acc[u]);
            }
        }
    }
    if (g < ng) {
        for (int u = 0; u < np; u++) {
            cd *ptr = Nbuf + (size_t)(slot * mlen + mm0 + u) * ldn + g;
            *ptr = cadd(*ptr, acc[u]);
        }
    }
}
