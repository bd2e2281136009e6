// dm_cluster.cuh -- DM iteration with one thread-block CLUSTER per frame (single probe mode), sm_100a.
//
// Same three passes as dm_mega.cuh, but the half-transformed frame never leaves the chip: a cluster of
// NCB CTAs works on one frame, CTA r owning row block r in passes 1 / 3 and column block r in pass 2.
// Pass 1 writes its row spectra straight into the COLUMN owners' shared memory (distributed shared
// memory, st.shared::cluster), pass 2 writes its result into the ROW owners' shared memory; two
// cluster barriers per frame replace the L2 ring, the per-slot flags and the release fences of the
// megakernel.  Clusters are persistent: cluster c takes slots c, c + nclusters, ...; a CTA's row block
// is fixed for the whole launch, so the lagged probe sums (reading R4) stay in registers until the end.
//
// Shared memory of one CTA: exchange of the line FFT, twiddles, colTile [N][LPB] (written by the
// cluster in pass 1, read here in pass 2), rowTile [LPB][N] (written by the cluster in pass 2, read
// here in pass 3), the frame's NCB error partials.  Buffer reuse is ordered by the two barriers:
//   colTile(f+1) is written after barrier B(f), by which every CTA has read colTile(f);
//   rowTile(f+1) and the partials are written after barrier A(f+1), by which every CTA has finished
//   pass 3 of frame f.
#pragma once
#include "dm_mega.cuh"

namespace ptycho {

__device__ __forceinline__ uint32_t cluster_rank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t map_to_rank(const void* local_smem, uint32_t rank) {   // address of the same object in CTA `rank`
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"((uint32_t)__cvta_generic_to_shared(local_smem)), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_cluster(uint32_t addr, float2 v) {
    asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(v.x), "f"(v.y) : "memory");
}
__device__ __forceinline__ void st_cluster(uint32_t addr, float v) {
    asm volatile("st.shared::cluster.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void cluster_sync() {     // release our (remote) stores, acquire everybody else's
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

template <int N> struct ClusterGeo {
    using G = Geo<N>;
    static constexpr int LINE = MegaGeo<N>::LINE;
    // exchange, twiddles (2N float4), colTile, rowTile, partials
    static constexpr size_t smem = (size_t)(G::LPB * LINE + 4 * N + 2 * G::LPB * N) * sizeof(float2) + 64 * sizeof(float);
};

struct ClusterArgs {
    FrameArgs f;            // psi = slot 0 of the store; e_part [J][NCB]
    int J, nclusters;
    int update_probe, det;
    const YX* spos;         // [J] positions in slot order
    const void* It;         // tiled intensities (k_tile_intensity)
};

template <int N, bool U16> __global__ void __launch_bounds__(kThreads, (N >= 512 ? 1 : 2)) k_dm_cluster(ClusterArgs m) {
    using G = Geo<N>;
    constexpr int E = G::E, T = G::T, LPB = G::LPB, NCB = G::NCB;
    const FrameArgs& a = m.f;
    extern __shared__ __align__(16) float2 sm[];
    float2* exch = sm;
    float4* s_tw = reinterpret_cast<float4*>(sm + LPB * ClusterGeo<N>::LINE);
    float2* colTile = reinterpret_cast<float2*>(s_tw + 2 * N);      // [N][LPB]
    float2* rowTile = colTile + LPB * N;                             // [LPB][N]
    float* s_err = reinterpret_cast<float*>(rowTile + LPB * N);      // [NCB] partials of the current frame
    __shared__ float s_red[kThreads / 32];
    load_tw(s_tw, a.tw, a.twi, N);
    const uint32_t rank = cluster_rank();
    const int cluster = blockIdx.x / NCB;
    // row passes: line l of row block `rank`; column pass: column c of column block `rank`
    const int l = threadIdx.x / T, t = threadIdx.x % T;
    const int c = threadIdx.x % LPB, tc = threadIdx.x / LPB;
    float2* sx_row = exch + l * G::LS_ROW;
    float2* sx_col = exch + c * G::LS_COL;
    const int y = rank * LPB + l;
    const size_t off = (size_t)y * N;
    constexpr float inv_n2 = 1.0f / ((float)N * (float)N);
    constexpr float kAmp2Floor = 1e-30f;
    const size_t tile_bytes = (size_t)N * LPB * (U16 ? 2 : 4);
    float2 accN[E];                                                  // lagged probe sums of ALL this CTA's frames (R4)
    float accD[E];
#pragma unroll
    for (int i = 0; i < E; ++i) { accN[i] = make_float2(0.f, 0.f); accD[i] = 0.f; }
    __syncthreads();
    cluster_sync();                                                  // every CTA of the cluster is resident before remote stores

    for (int slot = cluster; slot < m.J; slot += m.nclusters) {
        const YX p0 = m.spos[slot];
        {   // this CTA's rows of psi and its intensity tile for the cluster's NEXT frame: HBM -> L2 now
            const int nx = slot + m.nclusters;
            if (nx < m.J && (threadIdx.x & 31) == 0)
                l2_prefetch_bulk(a.psi + (size_t)nx * N * N + (size_t)(rank * LPB + (threadIdx.x >> 5) * (32 / T)) * N, (32 / T) * N * 8);
            if (nx < m.J && threadIdx.x == 32)
                l2_prefetch_bulk(reinterpret_cast<const char*>(m.It) + ((size_t)nx * NCB + rank) * tile_bytes, (uint32_t)tile_bytes);
        }
        // ---- pass 1: exit wave, reflector, probe sums, row FFTs -> column owners ---------------------
        {
            const float2* orow = a.O + (size_t)(p0.y + y) * a.W + p0.x;
            const float2* prow = a.psi + (size_t)slot * N * N + off;
            float2 v[E];
#pragma unroll
            for (int i = 0; i < E; ++i) v[i] = __ldcs(prow + t + T * i);
#pragma unroll
            for (int i = 0; i < E; ++i) {
                const float2 o = __ldg(orow + t + T * i);
                const float2 po = cmul(__ldg(a.P + off + t + T * i), o);
                const float2 s = v[i];
                if (m.update_probe) {
                    accN[i] = cadd(accN[i], cmulc(s, o));
                    accD[i] = fmaf(o.x, o.x, fmaf(o.y, o.y, accD[i]));
                }
                v[i] = make_float2(fmaf(2.f, po.x, -s.x), fmaf(2.f, po.y, -s.y));
            }
            fft_line_fwd<N, true>(v, t, sx_row, s_tw);
            __syncwarp();
#pragma unroll
            for (int r = 0; r < E; ++r) {                            // X[y][kx] -> colTile[y][kx % LPB] of CTA kx / LPB
                const int kx = freq_b<N>(t, r);
                st_cluster(map_to_rank(colTile + (size_t)y * LPB + kx % LPB, kx / LPB), v[r]);
            }
        }
        // intensities of pass 2: issued before the barrier, in flight while the cluster gathers
        constexpr int NQ = U16 ? E / 8 : E / 4;
        uint4 iq[NQ];
        {
            const uint4* it = reinterpret_cast<const uint4*>(reinterpret_cast<const char*>(m.It) + ((size_t)slot * NCB + rank) * tile_bytes) + threadIdx.x;
#pragma unroll
            for (int j = 0; j < NQ; ++j) iq[j] = __ldcs(it + j * kThreads);
        }
        cluster_sync();                                              // A: colTile complete
        // ---- pass 2: column FFTs, error partial, modulus projection (as s - 1), inverse columns -> row owners
        {
            float2 v[E];
#pragma unroll
            for (int i = 0; i < E; ++i) v[i] = colTile[(size_t)(tc + T * i) * LPB + c];
            fft_line_fwd<N>(v, tc, sx_col, s_tw);                    // (CTA barrier inside)
            float err = 0.f;
#pragma unroll
            for (int r = 0; r < E; ++r) {
                const float a2 = fmaf(v[r].x, v[r].x, v[r].y * v[r].y);
                const bool pos = a2 > kAmp2Floor;                    // R2
                const float ra = pos ? rsqrt_fast(a2) : 0.f;
                const float amp = a2 * ra;
                float inr;                                           // R3
                if (U16) {
                    const unsigned w = (&iq[r / 8].x)[(r % 8) / 2];
                    const unsigned u = (r & 1) ? (w >> 16) : (w & 0xffffu);
                    inr = u == 65535u ? -1.0f : (float)u;
                } else inr = __uint_as_float((&iq[r / 4].x)[r % 4]);
                if (inr >= 0.f) {
                    const float sq = sqrt_fast(inr), d = sq - amp;
                    err = fmaf(d, d, err);
                    if (pos) { const float sc = d * ra * inv_n2; v[r].x *= sc; v[r].y *= sc; }
                    else v[r] = make_float2(sq * inv_n2, 0.f);
                } else v[r] = make_float2(0.f, 0.f);
            }
#pragma unroll
            for (int s = 16; s > 0; s >>= 1) err += __shfl_xor_sync(0xffffffffu, err, s);
            if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = err;
            __syncthreads();                                         // exchange free again; s_red visible
            fft_line_inv<N>(v, tc, sx_col, s_tw + N);
            if (threadIdx.x < NCB) {                                 // this block's partial, fixed order, to every CTA of the cluster
                float tot = 0.f;
                for (int w = 0; w < kThreads / 32; ++w) tot += s_red[w];
                if (threadIdx.x == 0) a.e_part[(size_t)slot * NCB + rank] = tot;
                st_cluster(map_to_rank(s_err + rank, threadIdx.x), tot);
            }
            const int kx = rank * LPB + c;
#pragma unroll
            for (int r = 0; r < E; ++r) {                            // x[yy][kx] -> rowTile[yy % LPB][kx] of CTA yy / LPB
                const int yy = pos_a_inv<N>(tc, r);
                st_cluster(map_to_rank(rowTile + (size_t)(yy % LPB) * N + kx, yy / LPB), v[r]);
            }
        }
        cluster_sync();                                              // B: rowTile and the partials complete
        // ---- pass 3: inverse row FFTs, exit-wave update, object scatter-add -------------------------
        {
            float keep = 1.f;                                        // 1 - rb (R6)
            if (a.pbound > 0.f) {
                float e = 0.f;
                for (int i = 0; i < NCB; ++i) e += s_err[i];
                e *= inv_n2;
                keep = (e <= a.pbound) ? 0.f : 1.f - sqrtf(a.pbound / e);
            }
            const size_t obase = (size_t)(p0.y + y) * a.W + p0.x;
            float2 o[E];
#pragma unroll
            for (int r = 0; r < E; ++r) o[r] = __ldg(a.O + obase + pos_a_inv<N>(t, r));
            float2 v[E];
#pragma unroll
            for (int r = 0; r < E; ++r) v[r] = rowTile[(size_t)l * N + freq_b<N>(t, r)];
            fft_line_inv<N, true>(v, t, sx_row, s_tw + N);           // v = F^-1[(s-1) Phi]
            __syncwarp();
            float2* prow = a.psi + (size_t)slot * N * N + off;
#pragma unroll
            for (int r = 0; r < E; ++r) {
                const int x = pos_a_inv<N>(t, r);
                const float2 p = __ldg(a.P + off + x);
                const float2 po = cmul(p, o[r]);
                const float2 w = make_float2(fmaf(keep, v[r].x, po.x), fmaf(keep, v[r].y, po.y));
                __stcs(prow + x, w);
                if (!m.det) {
                    red_add(a.nO + obase + x, cmulc(w, p));
                    red_add(a.dO + obase + x, fmaf(p.x, p.x, p.y * p.y));
                }
            }
        }
        __syncthreads();                                             // the exchange is shared between the row and column views
    }
    if (m.update_probe) {
#pragma unroll
        for (int i = 0; i < E; ++i) {
            red_add(a.nP + off + t + T * i, accN[i]);
            red_add(a.dP + off + t + T * i, accD[i]);
        }
    }
    cluster_sync();                                                  // nobody exits while a neighbour may still write here
}

}  // namespace ptycho
