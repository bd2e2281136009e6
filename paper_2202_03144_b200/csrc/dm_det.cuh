// dm_det.cuh -- deterministic ("sorted-tile") accumulation of the DM overlap sums, sm_100a.
//
// north_star: "a tiled overlap accumulation with shared-memory pre-reduction before global atomics,
// plus a deterministic sorted-tile mode".  With ptycho_params.deterministic = 1 the DM megakernel
// does no floating-point atomics at all; the overlap sums of SURVEY.md 8(a) a8 / a9 are formed by two
// owner-computes kernels in which every output element adds its terms in ONE fixed order (slot
// order = the spatial sort fixed at init), so two runs give bit-identical O, P and psi:
//
//   k_det_probe  (before the megakernel: reading R4 wants the INCOMING psi_j and the current O)
//       n_P(r) = sum_j conj(O[r_j + r]) psi_j(r),  d_P(r) = sum_j |O[r_j + r]|^2
//       thread = one probe pixel; the J slots are cut into G fixed groups (grid.y), each group is
//       summed in slot order into partial[g][r]; k_det_probe_final adds the G partials in order.
//   k_det_object (after the megakernel: object sums want the NEW psi_j)
//       n_O(q) = sum_{j covers q} conj(P(q - r_j)) psi_j(q - r_j),  d_O(q) = sum |P(q - r_j)|^2
//       thread = one object pixel of a 32 x 8 tile; the tile's frame list (built on the host at
//       init, slot order) is walked in order.
//
// Cost: psi is read twice more (N^2 (32 K + b_I) bytes per pattern instead of N^2 (16 K + b_I)); the
// mode trades speed for reproducibility and bench.py times the atomic mode.
#pragma once
#include "kernels.cuh"

namespace ptycho {

constexpr int kDetTileW = 32, kDetTileH = 8;       // object tile of k_det_object (one pixel per thread)
constexpr int kDetGroups = 32;                     // frame groups of k_det_probe

// grid (n*n / 256, G).  partial: [G][n*n] float4 {Re n_P, Im n_P, d_P, 0}.
__global__ void __launch_bounds__(256) k_det_probe(float4* __restrict__ partial, const float2* __restrict__ psi,
                                                   const float2* __restrict__ O, int W, int n, const YX* __restrict__ spos, int J) {
    const int nn = n * n, q = blockIdx.x * 256 + threadIdx.x;
    if (q >= nn) return;
    const int y = q / n, x = q % n;
    const int per = (J + gridDim.y - 1) / gridDim.y;
    const int j0 = blockIdx.y * per, j1 = min(J, j0 + per);
    float2 an = make_float2(0.f, 0.f);
    float ad = 0.f;
    for (int j = j0; j < j1; ++j) {                                  // fixed order: slot order
        const YX p = spos[j];
        const float2 o = __ldg(O + (size_t)(p.y + y) * W + p.x + x);
        const float2 s = __ldcs(psi + (size_t)j * nn + q);
        an.x = fmaf(s.x, o.x, fmaf(s.y, o.y, an.x));                 // conj(o) * s
        an.y = fmaf(s.y, o.x, fmaf(-s.x, o.y, an.y));
        ad = fmaf(o.x, o.x, fmaf(o.y, o.y, ad));
    }
    partial[(size_t)blockIdx.y * nn + q] = make_float4(an.x, an.y, ad, 0.f);
}
// n_P, d_P = sum over the G groups, in group order.
__global__ void k_det_probe_final(float2* __restrict__ nP, float* __restrict__ dP, const float4* __restrict__ partial, int nn, int G) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= nn) return;
    float2 an = make_float2(0.f, 0.f);
    float ad = 0.f;
    for (int g = 0; g < G; ++g) {
        const float4 v = partial[(size_t)g * nn + q];
        an.x += v.x; an.y += v.y; ad += v.z;
    }
    nP[q] = an;
    dP[q] = ad;
}

// grid (tiles_x, tiles_y), block kDetTileW x kDetTileH.  tile_start[tile .. tile + 1] delimits the
// slots (ascending) whose frames overlap the tile.
__global__ void __launch_bounds__(kDetTileW * kDetTileH) k_det_object(float2* __restrict__ nO, float* __restrict__ dO, int H, int W,
                                                                       const float2* __restrict__ psi, const float2* __restrict__ P, int n,
                                                                       const YX* __restrict__ spos, const int* __restrict__ tile_start,
                                                                       const int* __restrict__ tile_list) {
    const int tile = blockIdx.y * gridDim.x + blockIdx.x;
    const int qx = blockIdx.x * kDetTileW + threadIdx.x, qy = blockIdx.y * kDetTileH + threadIdx.y;
    const int e0 = tile_start[tile], e1 = tile_start[tile + 1];
    const size_t nn = (size_t)n * n;
    float2 an = make_float2(0.f, 0.f);
    float ad = 0.f;
    for (int e = e0; e < e1; ++e) {                                  // fixed order: ascending slot
        const int j = tile_list[e];
        const YX p = spos[j];
        const int y = qy - p.y, x = qx - p.x;
        if (y < 0 || x < 0 || y >= n || x >= n) continue;
        const float2 pr = __ldg(P + (size_t)y * n + x);
        const float2 s = __ldcs(psi + (size_t)j * nn + (size_t)y * n + x);
        an.x = fmaf(s.x, pr.x, fmaf(s.y, pr.y, an.x));               // conj(P) * psi_j
        an.y = fmaf(s.y, pr.x, fmaf(-s.x, pr.y, an.y));
        ad = fmaf(pr.x, pr.x, fmaf(pr.y, pr.y, ad));
    }
    if (qy < H && qx < W) {
        nO[(size_t)qy * W + qx] = an;
        dO[(size_t)qy * W + qx] = ad;
    }
}

}  // namespace ptycho
