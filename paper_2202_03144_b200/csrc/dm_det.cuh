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

// a10 for the DM megakernel (dm_mega.cuh), which scatters only the CORRECTION term of the object sum:
// with psi'_j = P O_j + keep_j v_j (v_j = F^-1[(s - 1) Phi_j], keep_j = 1 - rb_j of the relaxed projection, R6),
//     n_O(q) = sum_j conj(P) psi'_j = d_O(q) O(q) + c(q),   c(q) = sum_j keep_j conj(P(q - r_j)) v_j(q - r_j),
// so the blended division of R5 becomes  O <- (n_O + eps O)/(d_O + eps) = O + c / (d_O + eps)  -- the same value, and frames whose
// error is already inside the power bound (keep_j = 0) add nothing.  d_O(q) = sum_j |P(q - r_j)|^2 depends only on the probe and
// the positions: it is gathered HERE over the tile's frame list instead of being scatter-added with one atomic per pixel and frame.
// Also zeroes c.
// |P|^2 table of the current probe; block 0 also rolls the megakernel's statistic: stat[0] <- frames inside the power bound in
// the iteration just run, stat[1] <- 0.
__global__ void __launch_bounds__(1024) k_probe_support(float* __restrict__ p2, const float2* __restrict__ P, int n, int* stat) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q < n * n) { const float2 v = P[q]; p2[q] = fmaf(v.x, v.x, v.y * v.y); }
    if (q == 0 && stat) { stat[0] = stat[1]; stat[1] = 0; }
}

// tile_start / tile_mid / tile_list: per 32 x 8 object tile, the packed positions (y << 16 | x) of the frames that overlap it,
// those covering the whole tile first ([tile_start, tile_mid)), then the partial ones ([tile_mid, tile_start[tile + 1])); each
// group in ascending slot order, so the sum has one fixed order.
__global__ void __launch_bounds__(kDetTileW * kDetTileH) k_dm_blend_gather(float2* __restrict__ O, float2* __restrict__ cO, int H, int W,
                                                                            const float* __restrict__ p2, int n, const int* __restrict__ tile_start,
                                                                            const int* __restrict__ tile_mid, const int* __restrict__ tile_list,
                                                                            const Scalars* __restrict__ sc) {
    constexpr int NT = kDetTileW * kDetTileH;
    __shared__ int s_off[NT];
    const int tile = blockIdx.y * gridDim.x + blockIdx.x, tid = threadIdx.y * kDetTileW + threadIdx.x;
    const int qx = blockIdx.x * kDetTileW + threadIdx.x, qy = blockIdx.y * kDetTileH + threadIdx.y;
    const int e0 = tile_start[tile], em = tile_mid[tile], e1 = tile_start[tile + 1];
    const bool in = qy < H && qx < W;
    const size_t i = (size_t)qy * W + qx;
    const float2 c = in ? cO[i] : make_float2(0.f, 0.f);
    // A tile whose correction is zero everywhere (every frame over it is inside its power bound: the steady state) keeps its
    // object values exactly; d_O is not needed there.
    if (!__syncthreads_or(c.x != 0.f || c.y != 0.f)) return;
    const float* pb = p2 + qy * n + qx;
    float d0 = 0.f, d1 = 0.f, d2 = 0.f, d3 = 0.f;
    for (int c0 = e0; c0 < em; c0 += NT) {                           // frames covering the whole tile: no per-pixel test, four loads in flight
        const int nc = min(NT, em - c0);
        __syncthreads();
        if (tid < nc) { const int v = tile_list[c0 + tid]; s_off[tid] = (v >> 16) * n + (v & 0xffff); }
        __syncthreads();
        int e = 0;
        for (; e + 4 <= nc; e += 4) {
            d0 += __ldg(pb - s_off[e]); d1 += __ldg(pb - s_off[e + 1]); d2 += __ldg(pb - s_off[e + 2]); d3 += __ldg(pb - s_off[e + 3]);
        }
        for (; e < nc; ++e) d0 += __ldg(pb - s_off[e]);
    }
    for (int c0 = em; c0 < e1; c0 += NT) {                           // frames covering part of it
        const int nc = min(NT, e1 - c0);
        __syncthreads();
        if (tid < nc) s_off[tid] = tile_list[c0 + tid];
        __syncthreads();
        for (int e = 0; e < nc; ++e) {
            const int y = qy - (s_off[e] >> 16), x = qx - (s_off[e] & 0xffff);
            if (y >= 0 && y < n && x >= 0 && x < n) d1 += __ldg(p2 + y * n + x);
        }
    }
    const float d = (d0 + d1) + (d2 + d3);
    if (!in) return;
    const float inv = 1.0f / (d + sc->eps_O);
    const float2 o = O[i];
    O[i] = make_float2(fmaf(c.x, inv, o.x), fmaf(c.y, inv, o.y));
    cO[i] = make_float2(0.f, 0.f);
}

}  // namespace ptycho
