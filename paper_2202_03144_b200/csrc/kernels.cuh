// kernels.cuh -- the projection-cycle kernels for sm_100a.
//
// Pipeline per chunk of frames ("three-pass, L2-resident"):
//   k_rows_fwd : a1 exit wave (+ a2 DM reflector, + DM lagged probe sums) fused into the load of
//                the row FFTs (a3, x direction); writes the half-transformed frame to scratch S.
//   k_cols     : column FFTs (a3, y direction), a4 per-frame error partials, a5 modulus
//                projection (exact scale; the relaxed blend is applied in k_rows_inv, which is
//                equivalent by linearity of F^-1), inverse column FFTs (a6), back to S.
//   k_rows_inv : inverse row FFTs (a6) fused with a7 exit-wave update and a8/a9 overlap
//                scatter-adds (vector red.global.add) of the object and probe sums.
// S is sized so that a chunk stays resident in the 126 MB L2; HBM sees psi in/out and I only.
#pragma once
#include <cstdint>
#include "fft_core.cuh"

namespace ptycho {

struct YX { int y, x; };

enum RowFwdMode { RF_EXIT = 0, RF_DM = 1, RF_PLAIN = 2, RF_EXIT_PJ = 3, RF_DM_PJ = 4 };   // _PJ: per-frame probes (sub-pixel positions, R28)
enum ColMode { CM_FULL = 0, CM_ERRONLY = 1, CM_PLAIN_FWD = 2, CM_PLAIN_INV = 3 };
enum RowInvMode { RI_MINIBATCH = 0, RI_DM = 1, RI_REVISED = 2, RI_PLAIN = 3, RI_LSQ_PF = 4, RI_MINIBATCH_PJ = 5, RI_DM_PJ = 6 };

#ifndef PTYCHO_THREADS
#define PTYCHO_THREADS 256
#endif
constexpr int kThreads = PTYCHO_THREADS;

struct FrameArgs {
    const float2* __restrict__ O;   // object H x W
    int W;
    const float2* __restrict__ P;   // K x N x N
    int K;
    float2* psi;                    // DM: exit-wave store of this launch's first slot (slot-major)
    const YX* __restrict__ pos;     // J positions, caller numbering
    const int* __restrict__ frames; // caller frame id of each slot of this launch
    float2* S;                      // scratch: nframes x K x N x N
    const void* __restrict__ I;     // intensities, caller numbering
    const void* __restrict__ It;    // intensities re-tiled per (DM slot, column block) in pass-2 register order (dm_mega.cuh)
    const int* __restrict__ slot_of; // caller frame -> DM slot (indexes It)
    int itype;                      // 0 f32, 1 u16
    float* e_part;                  // per slot: NCB error partials (this launch's first slot)
    float2* nO; float* dO;          // object canvases H x W
    float2* nP; float* dP;          // probe canvases K x N x N, N x N
    float pbound;
    float2* out;                    // RI_REVISED: nframes x K x N x N
    double* pf_part;                // RI_LSQ_PF: per slot of this launch, NCB x 5 partial sums (A11, A22, A12, b1, b2)
    const float2* __restrict__ tw;  // twiddles [ka*T + b]
    const float2* __restrict__ twi; // twiddles [b*E + ka]
    float2* Pj;                     // _PJ modes: this launch's per-frame probes P_jk = S_delta_j[P_k], nframes x K x N x N (like S); the
                                    // inverse row pass overwrites them with the probe terms conj(O_j) chi_jk (R28)
    float2* Gj;                     // RF_DM_PJ: the lagged probe terms conj(O_j) psi_jk of this launch's frames, kept per frame (shifted back later)
};

template <int N> struct Geo {
    static constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T;
    static constexpr int LPB = kThreads / T;                     // lines per CTA
    static constexpr int LS_ROW = LineSmem<N>::SIZE + ((T == 8 && (LineSmem<N>::SIZE % 16) != 8) ? 8 : 0);
    static constexpr int LS_COL = LineSmem<N>::SIZE | 1;         // odd: lanes run along lines
    static constexpr int NCB = N / LPB;                          // column blocks (= row blocks) per frame
    static constexpr size_t smem_rows = (size_t)(LPB * LS_ROW + 2 * N * kTwWords) * sizeof(float2);
    static size_t smem_cols(int K) {
        (void)K;
        return (size_t)(LPB * LS_COL + 2 * N * kTwWords) * sizeof(float2) + 64;
    }
};

// Twiddle tables in shared memory, packed for the two-wide multiply (fft_core.cuh tw_pack): 2 n float4.
__device__ __forceinline__ void load_tw(tw_t* s_tw, const float2* tw, const float2* twi, int n) {
    for (int i = threadIdx.x; i < n; i += kThreads) { s_tw[i] = tw_store(tw[i], s_tw); s_tw[n + i] = tw_store(twi[i], s_tw); }
}

__device__ __forceinline__ float load_intensity(const void* I, int itype, size_t idx) {
    if (itype == 1) {
        const unsigned short v = __ldg(reinterpret_cast<const unsigned short*>(I) + idx);
        return v == 65535 ? -1.0f : (float)v;
    }
    return __ldg(reinterpret_cast<const float*>(I) + idx);
}

__device__ __forceinline__ void red_add(float2* p, float2 v) { atomicAdd(p, v); }
__device__ __forceinline__ void red_add(float* p, float v) { atomicAdd(p, v); }

// ------------------------------------------------------------------------------------------
// a1/a2/a3: exit wave (+ reflector) -> forward row FFTs -> S.   grid (NCB, nframes)
// ------------------------------------------------------------------------------------------
template <int N, int MODE> __global__ void __launch_bounds__(kThreads) k_rows_fwd(FrameArgs a) {
    using G = Geo<N>;
    constexpr int E = G::E, T = G::T;
    extern __shared__ __align__(16) float2 sm[];
    tw_t* s_tw = reinterpret_cast<tw_t*>(sm + G::LPB * G::LS_ROW);
    load_tw(s_tw, a.tw, a.twi, N);
    const int l = threadIdx.x / T, t = threadIdx.x % T;
    float2* sx = sm + l * G::LS_ROW;
    const int slot = blockIdx.y, y = blockIdx.x * G::LPB + l;
    const size_t fr = (size_t)slot * a.K * N * N;
    __syncthreads();

    if (MODE == RF_PLAIN) {
        float2 v[E];
        float2* row = a.S + fr + (size_t)y * N;
#pragma unroll
        for (int i = 0; i < E; ++i) v[i] = row[t + T * i];
        fft_line_fwd<N>(v, t, sx, s_tw);
#pragma unroll
        for (int r = 0; r < E; ++r) row[freq_b<N>(t, r)] = v[r];
        return;
    }

    const YX p0 = a.pos[a.frames[slot]];
    const float2* orow = a.O + (size_t)(p0.y + y) * a.W + p0.x;
    float2 o[E];
#pragma unroll
    for (int i = 0; i < E; ++i) o[i] = __ldg(orow + t + T * i);
    for (int k = 0; k < a.K; ++k) {
        const size_t off = ((size_t)k * N + y) * N;
        float2 v[E];
#pragma unroll
        for (int i = 0; i < E; ++i) v[i] = cmul((MODE == RF_EXIT_PJ || MODE == RF_DM_PJ) ? a.Pj[fr + off + t + T * i] : __ldg(a.P + off + t + T * i), o[i]);   // psi_O = P_k O_j
        if (MODE == RF_DM || MODE == RF_DM_PJ) {
            const float2* prow = a.psi + fr + off;
#pragma unroll
            for (int i = 0; i < E; ++i) {
                const float2 s = prow[t + T * i];
                if (MODE == RF_DM_PJ) a.Gj[fr + off + t + T * i] = cmulc(s, o[i]);      // kept per frame: shifted back before it is summed (R28)
                else red_add(a.nP + off + t + T * i, cmulc(s, o[i]));                   // conj(O_j) psi_j (lagged, R4)
                v[i] = make_float2(2.f * v[i].x - s.x, 2.f * v[i].y - s.y);             // reflector
            }
        }
        fft_line_fwd<N, true>(v, t, sx, s_tw);          // a row's T threads sit in one warp
        float2* srow = a.S + fr + off;
#pragma unroll
        for (int r = 0; r < E; ++r) srow[freq_b<N>(t, r)] = v[r];
        __syncwarp();
    }
    if (MODE == RF_DM || MODE == RF_DM_PJ) {
#pragma unroll
        for (int i = 0; i < E; ++i) red_add(a.dP + (size_t)y * N + t + T * i, o[i].x * o[i].x + o[i].y * o[i].y);
    }
}

// ------------------------------------------------------------------------------------------
// a3 (columns) / a4 / a5 / a6 (columns).   grid (NCB, nframes); CTA = LPB columns x T threads,
// lanes run along the columns so that every global access is LPB*8 contiguous bytes.
// ------------------------------------------------------------------------------------------
template <int N, int MODE> __global__ void __launch_bounds__(kThreads) k_cols(FrameArgs a) {
    using G = Geo<N>;
    constexpr int E = G::E, T = G::T, CB = G::LPB;
    extern __shared__ __align__(16) float2 sm[];
    tw_t* s_tw = reinterpret_cast<tw_t*>(sm + CB * G::LS_COL);
    __shared__ float s_red[kThreads / 32];
    load_tw(s_tw, a.tw, a.twi, N);
    const int c = threadIdx.x % CB, t = threadIdx.x / CB;
    float2* sx = sm + c * G::LS_COL;
    const int slot = blockIdx.y, col = blockIdx.x * CB + c;
    const size_t fr = (size_t)slot * a.K * N * N;
    __syncthreads();

    if (MODE == CM_PLAIN_FWD || MODE == CM_PLAIN_INV) {
        float2 v[E];
        float2* base = a.S + fr + col;
        if (MODE == CM_PLAIN_FWD) {
#pragma unroll
            for (int i = 0; i < E; ++i) v[i] = base[(size_t)(t + T * i) * N];
            fft_line_fwd<N>(v, t, sx, s_tw);
#pragma unroll
            for (int r = 0; r < E; ++r) base[(size_t)freq_b<N>(t, r) * N] = v[r];
        } else {
#pragma unroll
            for (int r = 0; r < E; ++r) v[r] = base[(size_t)freq_b<N>(t, r) * N];
            fft_line_inv<N>(v, t, sx, s_tw + N);
#pragma unroll
            for (int r = 0; r < E; ++r) base[(size_t)pos_a_inv<N>(t, r) * N] = v[r];
        }
        return;
    }

    float amp2[E];
#pragma unroll
    for (int r = 0; r < E; ++r) amp2[r] = 0.f;
    float2 v[E];
    for (int k = 0; k < a.K; ++k) {
        const float2* base = a.S + fr + (size_t)k * N * N + col;
#pragma unroll
        for (int i = 0; i < E; ++i) v[i] = base[(size_t)(t + T * i) * N];
        fft_line_fwd<N>(v, t, sx, s_tw);
#pragma unroll
        for (int r = 0; r < E; ++r) amp2[r] += v[r].x * v[r].x + v[r].y * v[r].y;
        if (a.K > 1) {
#pragma unroll
            for (int r = 0; r < E; ++r) const_cast<float2*>(base)[(size_t)freq_b<N>(t, r) * N] = v[r];   // K > 1: the spectrum waits in S (L2), not in shared memory: keeps 2-3 CTAs per SM
        }
        __syncthreads();
    }
    // I_j in this thread's register order: 16-byte chunks of the tiled copy (dm_mega.cuh k_tile_intensity)
    float in_t[E];
    {
        const size_t tile_bytes = (size_t)N * CB * (a.itype == 1 ? 2 : 4);
        const uint4* it = reinterpret_cast<const uint4*>(reinterpret_cast<const char*>(a.It) +
                                                         ((size_t)a.slot_of[a.frames[slot]] * G::NCB + blockIdx.x) * tile_bytes) + threadIdx.x;
        if (a.itype == 1) {
#pragma unroll
            for (int j = 0; j < E / 8; ++j) {
                const uint4 q = __ldg(it + j * kThreads);
                const unsigned w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const unsigned lo = w[k] & 0xffffu, hi = w[k] >> 16;
                    in_t[8 * j + 2 * k] = lo == 65535u ? -1.0f : (float)lo;
                    in_t[8 * j + 2 * k + 1] = hi == 65535u ? -1.0f : (float)hi;
                }
            }
        } else {
#pragma unroll
            for (int j = 0; j < E / 4; ++j) {
                const float4 q = __ldg(reinterpret_cast<const float4*>(it) + j * kThreads);
                in_t[4 * j] = q.x; in_t[4 * j + 1] = q.y; in_t[4 * j + 2] = q.z; in_t[4 * j + 3] = q.w;
            }
        }
    }
    // a4 error term and a5 scale.  scale[r] carries the 1/N^2 of F^-1.
    constexpr float inv_n2 = 1.0f / ((float)N * (float)N);
    float err = 0.f;
    float scale[E];
    bool zero_amp = false;
#pragma unroll
    for (int r = 0; r < E; ++r) {
        const float in = in_t[r];
        const float amp = sqrtf(amp2[r]);
        if (in >= 0.f) {
            const float sq = sqrtf(in), d = sq - amp;
            err = fmaf(d, d, err);
            if (amp2[r] > 1e-30f) scale[r] = sq / amp * inv_n2;   // R2 threshold shared with dm_mega.cuh: below it |Phi| counts as 0
            else { scale[r] = -sq * inv_n2; zero_amp = true; }   // R2: flagged by the sign
        } else scale[r] = inv_n2;                                 // R3: masked, keep Phi
    }
    // block reduction of the error partial (fixed order: deterministic)
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) err += __shfl_xor_sync(0xffffffffu, err, s);
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = err;
    __syncthreads();
    if (threadIdx.x == 0) {
        float tot = 0.f;
        for (int w = 0; w < kThreads / 32; ++w) tot += s_red[w];
        a.e_part[(size_t)slot * G::NCB + blockIdx.x] = tot;
    }
    if (MODE == CM_ERRONLY) return;

    for (int k = 0; k < a.K; ++k) {
        if (a.K > 1) {
#pragma unroll
            for (int r = 0; r < E; ++r) v[r] = (a.S + fr + (size_t)k * N * N + col)[(size_t)freq_b<N>(t, r) * N];   // this thread's own stores
        }
#pragma unroll
        for (int r = 0; r < E; ++r) {
            if (zero_amp && scale[r] < 0.f) v[r] = make_float2(k == 0 ? -scale[r] : 0.f, 0.f);
            else { v[r].x *= scale[r]; v[r].y *= scale[r]; }
        }
        fft_line_inv<N>(v, t, sx, s_tw + N);
        float2* base = a.S + fr + (size_t)k * N * N + col;
#pragma unroll
        for (int r = 0; r < E; ++r) base[(size_t)pos_a_inv<N>(t, r) * N] = v[r];
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------
// a6 (rows) / a7 / a8 / a9: inverse row FFTs -> revised wave -> exit-wave update -> scatter-add.
// grid (NCB, nframes)
// ------------------------------------------------------------------------------------------
template <int N, int MODE> __global__ void __launch_bounds__(kThreads, (N >= 512 ? 1 : 2)) k_rows_inv(FrameArgs a) {
    using G = Geo<N>;
    constexpr int E = G::E, T = G::T;
    extern __shared__ __align__(16) float2 sm[];
    tw_t* s_tw = reinterpret_cast<tw_t*>(sm + G::LPB * G::LS_ROW);
    load_tw(s_tw, a.tw, a.twi, N);
    const int l = threadIdx.x / T, t = threadIdx.x % T;
    float2* sx = sm + l * G::LS_ROW;
    const int slot = blockIdx.y, y = blockIdx.x * G::LPB + l;
    const size_t fr = (size_t)slot * a.K * N * N;
    __syncthreads();

    if (MODE == RI_PLAIN) {
        float2 v[E];
        float2* row = a.S + fr + (size_t)y * N;
#pragma unroll
        for (int r = 0; r < E; ++r) v[r] = row[freq_b<N>(t, r)];
        fft_line_inv<N>(v, t, sx, s_tw + N);
#pragma unroll
        for (int r = 0; r < E; ++r) row[pos_a_inv<N>(t, r)] = v[r];
        return;
    }

    // R6 relaxed projection: blend weight of this frame from its error partials (fixed order)
    float rb = 0.f;
    if (a.pbound > 0.f) {
        float e = 0.f;
        for (int i = 0; i < G::NCB; ++i) e += a.e_part[(size_t)slot * G::NCB + i];
        e *= 1.0f / ((float)N * (float)N);
        rb = (e <= a.pbound) ? 1.0f : sqrtf(a.pbound / e);
    }
    const YX p0 = a.pos[a.frames[slot]];
    const size_t obase = (size_t)(p0.y + y) * a.W + p0.x;
    float2 o[E];
#pragma unroll
    for (int r = 0; r < E; ++r) o[r] = __ldg(a.O + obase + pos_a_inv<N>(t, r));
    float2 accO[E];
    float accD[E];
    float pfs[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int r = 0; r < E; ++r) { accO[r] = make_float2(0.f, 0.f); accD[r] = 0.f; }

    for (int k = 0; k < a.K; ++k) {
        const size_t off = ((size_t)k * N + y) * N;
        float2 v[E];
        const float2* srow = a.S + fr + off;
#pragma unroll
        for (int r = 0; r < E; ++r) v[r] = srow[freq_b<N>(t, r)];
        fft_line_inv<N, true>(v, t, sx, s_tw + N);      // v = F^-1[exact projection]
#pragma unroll
        for (int r = 0; r < E; ++r) {
            const int x = pos_a_inv<N>(t, r);
            const float2 p = (MODE == RI_MINIBATCH_PJ || MODE == RI_DM_PJ) ? a.Pj[fr + off + x] : __ldg(a.P + off + x);
            const float2 po = cmul(p, o[r]);            // psi_O
            float2 w;
            if (MODE == RI_DM || MODE == RI_DM_PJ) {
                float2* ps = a.psi + fr + off + x;
                const float2 s = *ps;
                const float2 phi = make_float2(2.f * po.x - s.x, 2.f * po.y - s.y);
                const float2 pf = make_float2(fmaf(rb, phi.x - v[r].x, v[r].x), fmaf(rb, phi.y - v[r].y, v[r].y));
                w = make_float2(s.x + pf.x - po.x, s.y + pf.y - po.y);     // a7, beta = 1
                *ps = w;
            } else {
                const float2 pf = make_float2(fmaf(rb, po.x - v[r].x, v[r].x), fmaf(rb, po.y - v[r].y, v[r].y));
                if (MODE == RI_REVISED) { a.out[fr + off + x] = pf; continue; }
                w = make_float2(pf.x - po.x, pf.y - po.y);                 // chi
                if (MODE == RI_LSQ_PF) {                                   // R25: this frame's five sums; nO / nP hold the directions dO / dP_k
                    const float2 u = cmul(p, a.nO[obase + x]), vv = cmul(a.nP[off + x], o[r]);
                    pfs[0] = fmaf(u.x, u.x, fmaf(u.y, u.y, pfs[0]));
                    pfs[1] = fmaf(vv.x, vv.x, fmaf(vv.y, vv.y, pfs[1]));
                    pfs[2] = fmaf(u.x, vv.x, fmaf(u.y, vv.y, pfs[2]));
                    pfs[3] = fmaf(u.x, w.x, fmaf(u.y, w.y, pfs[3]));
                    pfs[4] = fmaf(vv.x, w.x, fmaf(vv.y, w.y, pfs[4]));
                    continue;
                }
                if (MODE == RI_MINIBATCH_PJ) a.Pj[fr + off + x] = cmulc(w, o[r]);   // kept per frame: shifted back before it is summed (R28)
                else red_add(a.nP + off + x, cmulc(w, o[r]));              // a9 conj(O_j) chi
            }
            accO[r] = cadd(accO[r], cmulc(w, p));                          // a8 conj(P_k) w
            accD[r] = fmaf(p.x, p.x, fmaf(p.y, p.y, accD[r]));
        }
        __syncwarp();
    }
    if (MODE == RI_REVISED) return;
    if (MODE == RI_LSQ_PF) {                                               // block reduction in a fixed order, in double
        __shared__ double s_pf[kThreads / 32][5];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
            double d = (double)pfs[q];
            for (int sft = 16; sft > 0; sft >>= 1) d += __shfl_xor_sync(0xffffffffu, d, sft);
            if ((threadIdx.x & 31) == 0) s_pf[threadIdx.x >> 5][q] = d;
        }
        __syncthreads();
        if (threadIdx.x < 5) {
            double d = 0.0;
            for (int wv = 0; wv < kThreads / 32; ++wv) d += s_pf[wv][threadIdx.x];
            a.pf_part[((size_t)slot * G::NCB + blockIdx.x) * 5 + threadIdx.x] = d;
        }
        return;
    }
#pragma unroll
    for (int r = 0; r < E; ++r) {
        const int x = pos_a_inv<N>(t, r);
        red_add(a.nO + obase + x, accO[r]);
        red_add(a.dO + obase + x, accD[r]);
        if (MODE == RI_MINIBATCH || MODE == RI_MINIBATCH_PJ) red_add(a.dP + (size_t)y * N + x, o[r].x * o[r].x + o[r].y * o[r].y);
    }
}

// ------------------------------------------------------------------------------------------
// small element-wise / reduction kernels (a10, a11)
// ------------------------------------------------------------------------------------------
// psi_j = P O_j for every slot (R4 initial exit waves).  grid (nslots, N*N*K / 256)
__global__ void k_init_psi(float2* psi, const float2* __restrict__ O, int W, const float2* __restrict__ P, int K,
                           int n, const YX* __restrict__ pos, const int* __restrict__ frames) {
    const int slot = blockIdx.x;
    const size_t i = (size_t)blockIdx.y * blockDim.x + threadIdx.x;   // over K*n*n
    const size_t nn = (size_t)n * n;
    if (i >= nn * K) return;
    const size_t q = i % nn;
    const int y = (int)(q / n), x = (int)(q % n);
    const YX p0 = pos[frames[slot]];
    psi[(size_t)slot * K * nn + i] = cmul(P[i], O[(size_t)(p0.y + y) * W + p0.x + x]);
}

// gather stored exit waves of listed slots into out (fetch) or scatter from in (set)
__global__ void k_copy_frames(float2* dst, const float2* src, const int* __restrict__ dst_idx,
                              const int* __restrict__ src_idx, size_t per_frame) {
    const size_t d = dst_idx ? (size_t)dst_idx[blockIdx.y] : blockIdx.y;
    const size_t s = src_idx ? (size_t)src_idx[blockIdx.y] : blockIdx.y;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < per_frame; i += (size_t)gridDim.x * blockDim.x)
        dst[d * per_frame + i] = src[s * per_frame + i];
}

struct Scalars {            // device-resident scalars (no host round trip inside iterate)
    float max_p2;           // max_r sum_k |P_k|^2 of the current probe
    float max_dp;           // max_r d_P of the current batch
    float step_a, step_b;   // steps applied by the apply kernels
    double sum_I;           // sum of unmasked intensities of the frames present
    double sum_I_iter;      // its value when the running iteration started (frames may be appended meanwhile)
    float eps_O, eps_P;     // DM blend constants (fixed at init)
    float max_p2s[2];       // ePIE-minibatch: max_r sum_k |P_k|^2 of the probe the NEXT batch starts from, ping-pong (k_epie_update)
    unsigned int max_bits;  // scratch for atomicMax on non-negative floats
};

// max over r of sum_k |P_k(r)|^2 -> sc->max_p2 (zeroed by the caller; atomicMax on the bit pattern of
// non-negative floats is order-independent, hence deterministic).
__global__ void k_probe_max(const float2* __restrict__ P, int K, int nn, Scalars* sc) {
    float m = 0.f;
    for (int q = blockIdx.x * blockDim.x + threadIdx.x; q < nn; q += gridDim.x * blockDim.x) {
        float v = 0.f;
        for (int k = 0; k < K; ++k) { const float2 p = P[(size_t)k * nn + q]; v += p.x * p.x + p.y * p.y; }
        m = fmaxf(m, v);
    }
    for (int d = 16; d > 0; d >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, d));
    if ((threadIdx.x & 31) == 0) atomicMax(reinterpret_cast<unsigned int*>(&sc->max_p2), __float_as_uint(m));
}
// max over r of d_P(r) -> sc->max_dp (zeroed by the caller).
__global__ void k_real_max(const float* __restrict__ d, int nn, Scalars* sc) {
    float m = 0.f;
    for (int q = blockIdx.x * blockDim.x + threadIdx.x; q < nn; q += gridDim.x * blockDim.x) m = fmaxf(m, d[q]);
    for (int dd = 16; dd > 0; dd >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, dd));
    if ((threadIdx.x & 31) == 0) atomicMax(reinterpret_cast<unsigned int*>(&sc->max_dp), __float_as_uint(m));
}
// max |O|^2 at init (for eps_P); uses atomicMax on the bit pattern of non-negative floats.
__global__ void k_abs2_max(const float2* __restrict__ a, size_t n, Scalars* sc) {
    float m = 0.f;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        m = fmaxf(m, a[i].x * a[i].x + a[i].y * a[i].y);
    for (int d = 16; d > 0; d >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, d));
    if ((threadIdx.x & 31) == 0) atomicMax(&sc->max_bits, __float_as_uint(m));
}

// a10 DM: x <- (n + eps x)/(d + eps); zero the canvases.  which = 0 object (eps_O), 1 probe (eps_P);
// d is shared by the `modes` planes of n.
__global__ void k_dm_blend(float2* x, float2* n, float* d, size_t plane, int modes, const Scalars* sc, int which,
                           int update) {
    const float eps = which ? sc->eps_P : sc->eps_O;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < plane; i += (size_t)gridDim.x * blockDim.x) {
        const float inv = 1.0f / (d[i] + eps);
        for (int k = 0; k < modes; ++k) {
            const size_t q = (size_t)k * plane + i;
            if (update) { const float2 xv = x[q], nv = n[q]; x[q] = make_float2((nv.x + eps * xv.x) * inv, (nv.y + eps * xv.y) * inv); }
            n[q] = make_float2(0.f, 0.f);
        }
        d[i] = 0.f;
    }
}

// minibatch directions: n <- n / (d + delta * max)  (in place), optional LSQML partial sums
//   part[2*block + 0] += sum |dir|^2 d     (A11 or A22)
//   part[2*block + 1] += sum Re conj(dir) n_before   (b1 or b2)
// which = 0: object (max = max_p2), 1: probe (max = max_dp).
__global__ void k_direction(float2* n, const float* __restrict__ d, size_t plane, int modes, float delta,
                            const Scalars* sc, int which, double* part) {
    const float reg = delta * (which ? sc->max_dp : sc->max_p2);
    double a = 0.0, b = 0.0;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    // four pixels per thread and step, loads first: one 8-byte load in flight per thread kept this kernel at half the HBM rate
    for (; i + 3 * stride < plane; i += 4 * stride) {
        float dv[4], inv[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) dv[u] = d[i + u * stride];
#pragma unroll
        for (int u = 0; u < 4; ++u) inv[u] = 1.0f / (dv[u] + reg);
        for (int k = 0; k < modes; ++k) {
            float2 nv[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) nv[u] = n[(size_t)k * plane + i + u * stride];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float2 dir = make_float2(nv[u].x * inv[u], nv[u].y * inv[u]);
                n[(size_t)k * plane + i + u * stride] = dir;
                if (part) {
                    a += (double)((dir.x * dir.x + dir.y * dir.y) * dv[u]);
                    b += (double)(dir.x * nv[u].x + dir.y * nv[u].y);
                }
            }
        }
    }
    for (; i < plane; i += stride) {
        const float dv = d[i], inv = 1.0f / (dv + reg);
        for (int k = 0; k < modes; ++k) {
            const size_t q = (size_t)k * plane + i;
            const float2 nv = n[q];
            const float2 dir = make_float2(nv.x * inv, nv.y * inv);
            n[q] = dir;
            if (part) {
                a += (double)((dir.x * dir.x + dir.y * dir.y) * dv);
                b += (double)(dir.x * nv.x + dir.y * nv.y);
            }
        }
    }
    if (part) {
        __shared__ double sa[32], sb[32];
        for (int s = 16; s > 0; s >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, s); b += __shfl_xor_sync(0xffffffffu, b, s); }
        if ((threadIdx.x & 31) == 0) { sa[threadIdx.x >> 5] = a; sb[threadIdx.x >> 5] = b; }
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int w = 1; w < (int)blockDim.x / 32; ++w) { a += sa[w]; b += sb[w]; }
            part[2 * blockIdx.x] = a; part[2 * blockIdx.x + 1] = b;
        }
    }
}

// LSQML cross term A12 = Re sum_j sum_r T(r) conj(dO[r_j+r]) O[r_j+r],  T = sum_k conj(P_k) dP_k.
// grid (nframes, parts): block (f, p) sums every parts-th pixel group of frame f; part[f * parts + p].
// T = sum_k conj(P_k) dP_k, the same for every frame of the batch: formed once (k_lsq_T), gathered by k_lsq_cross.
__global__ void k_lsq_T(float2* __restrict__ T, const float2* __restrict__ P, const float2* __restrict__ dPk, int K, int nn) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= nn) return;
    float2 tq = make_float2(0.f, 0.f);
    for (int k = 0; k < K; ++k) tq = cadd(tq, cmulc(dPk[(size_t)k * nn + q], P[(size_t)k * nn + q]));
    T[q] = tq;
}
__global__ void k_lsq_cross(const float2* __restrict__ O, const float2* __restrict__ dO, int W, const float2* __restrict__ T, int n, int log2n,
                            const YX* __restrict__ pos, const int* __restrict__ frames, double* part) {
    const YX p0 = pos[frames[blockIdx.x]];
    const int nn = n * n, stride = gridDim.y * blockDim.x;
    const size_t base = (size_t)p0.y * W + p0.x;
    double acc = 0.0;
    int q = blockIdx.y * blockDim.x + threadIdx.x;
    for (; q + 3 * stride < nn; q += 4 * stride) {          // four gathers in flight (n is a power of two: no division)
        float2 t[4], o[4], d[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int qq = q + u * stride;
            const size_t i = base + (size_t)(qq >> log2n) * W + (qq & (n - 1));
            t[u] = __ldg(T + qq); o[u] = __ldg(O + i); d[u] = __ldg(dO + i);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const float2 s = cmulc(o[u], d[u]);            // conj(dO) O
            acc += (double)(t[u].x * s.x - t[u].y * s.y);
        }
    }
    for (; q < nn; q += stride) {
        const size_t i = base + (size_t)(q >> log2n) * W + (q & (n - 1));
        const float2 s = cmulc(O[i], dO[i]);
        acc += (double)(T[q].x * s.x - T[q].y * s.y);
    }
    __shared__ double sa[32];
    for (int s = 16; s > 0; s >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, s);
    if ((threadIdx.x & 31) == 0) sa[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) { for (int w = 1; w < (int)blockDim.x / 32; ++w) acc += sa[w]; part[blockIdx.x * gridDim.y + blockIdx.y] = acc; }
}

// a11: sum the partials in a fixed order (thread-strided, then a shared-memory tree: the same order
// on every run), solve the 2x2 system (R9), publish the steps.  One CTA of 256 threads.
// partA22 != nullptr (sub-pixel positions, R28): A22 comes from the per-frame sums of k_lsq_cross_pj instead of the canvas closed form.
__global__ void k_lsq_solve(const double* partO, int nO, const double* partP, int nP, const double* partX, int nX,
                            float lambda, int update_probe, Scalars* sc, double* steps_out, const double* partA22 = nullptr) {
    __shared__ double sh[5][256];
    double v[5] = {0, 0, 0, 0, 0};                       // A11, b1, A22, b2, A12
    for (int i = threadIdx.x; i < nO; i += 256) { v[0] += partO[2 * i]; v[1] += partO[2 * i + 1]; }
    for (int i = threadIdx.x; i < nP; i += 256) { if (!partA22) v[2] += partP[2 * i]; v[3] += partP[2 * i + 1]; }
    for (int i = threadIdx.x; i < nX; i += 256) { v[4] += partX[i]; if (partA22) v[2] += partA22[i]; }
    for (int q = 0; q < 5; ++q) sh[q][threadIdx.x] = v[q];
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if ((int)threadIdx.x < w)
            for (int q = 0; q < 5; ++q) sh[q][threadIdx.x] += sh[q][threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x) return;
    const double A11 = sh[0][0], b1 = sh[1][0], A22 = sh[2][0], b2 = sh[3][0], A12 = sh[4][0];
    const double l = 1.0 + (double)lambda;
    double a, b;
    if (!update_probe) { a = (A11 > 0) ? b1 / (A11 * l) : 0.0; b = 0.0; }
    else {
        const double det = A11 * l * A22 * l - A12 * A12;
        if (!(det > 0) || !isfinite(det)) { a = 0; b = 0; }
        else { a = (b1 * A22 * l - A12 * b2) / det; b = (A11 * l * b2 - A12 * b1) / det; }
    }
    sc->step_a = (float)a; sc->step_b = (float)b;
    steps_out[0] = a; steps_out[1] = b;
}
// R25: per-frame 2x2 solves from the partial sums of RI_LSQ_PF (NCB x 5 per frame, added in block order), one CTA; the probe
// step is the mean b_j (fixed-order tree).  ab: nb x (a_j, b_j) floats for the scatter; steps_out (optional): the same pairs, double.
__global__ void __launch_bounds__(1024) k_lsq_pf_solve(const double* __restrict__ part, int nb, int ncb, float lambda, int update_probe, float2* ab,
                                                       Scalars* sc, double* steps_out, int steps_cap) {
    __shared__ double sb[1024];
    const double l = 1.0 + (double)lambda;
    double bsum = 0.0;
    for (int j = threadIdx.x; j < nb; j += 1024) {
        double v[5] = {0, 0, 0, 0, 0};
        for (int b = 0; b < ncb; ++b)
            for (int q = 0; q < 5; ++q) v[q] += part[((size_t)j * ncb + b) * 5 + q];
        const double A11 = v[0], A22 = v[1], A12 = v[2], b1 = v[3], b2 = v[4];
        double a, b;
        if (!update_probe) { a = (A11 > 0) ? b1 / (A11 * l) : 0.0; b = 0.0; }
        else {
            const double det = A11 * l * A22 * l - A12 * A12;
            if (!(det > 0) || !isfinite(det)) { a = 0; b = 0; }
            else { a = (b1 * A22 * l - A12 * b2) / det; b = (A11 * l * b2 - A12 * b1) / det; }
        }
        ab[j] = make_float2((float)a, (float)b);
        if (steps_out && j < steps_cap) { steps_out[2 * j] = a; steps_out[2 * j + 1] = b; }
        bsum += b;
    }
    sb[threadIdx.x] = bsum;
    __syncthreads();
    for (int w = 512; w > 0; w >>= 1) { if ((int)threadIdx.x < w) sb[threadIdx.x] += sb[threadIdx.x + w]; __syncthreads(); }
    if (threadIdx.x == 0) { sc->step_a = 1.f; sc->step_b = (float)(sb[0] / nb); }
}
// R25 weighted second scatter: aw += a_j w_j, ww += w_j, w_j = sum_k |P_k|^2 on the frame's window.  grid (nframes, n*n/256)
__global__ void k_lsq_pf_scatter(float* aw, float* ww, int W, const float2* __restrict__ P, int K, int n, const YX* __restrict__ pos,
                                 const int* __restrict__ frames, const float2* __restrict__ ab) {
    const int q = blockIdx.y * blockDim.x + threadIdx.x, nn = n * n;
    if (q >= nn) return;
    const YX p0 = pos[frames[blockIdx.x]];
    float w = 0.f;
    for (int k = 0; k < K; ++k) { const float2 p = P[(size_t)k * nn + q]; w = fmaf(p.x, p.x, fmaf(p.y, p.y, w)); }
    const size_t o = (size_t)(p0.y + q / n) * W + p0.x + q % n;
    atomicAdd(aw + o, ab[blockIdx.x].x * w);
    atomicAdd(ww + o, w);
}
// O += dO * aw / ww where ww > 0; zero dO (dir), aw, ww.
__global__ void k_lsq_pf_apply(float2* x, float2* dir, float* aw, float* ww, size_t plane) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < plane; i += (size_t)gridDim.x * blockDim.x) {
        const float wv = ww[i];
        if (wv > 0.f) { const float st = aw[i] / wv; const float2 d = dir[i]; float2 xv = x[i]; xv.x = fmaf(st, d.x, xv.x); xv.y = fmaf(st, d.y, xv.y); x[i] = xv; }
        dir[i] = make_float2(0.f, 0.f); aw[i] = 0.f; ww[i] = 0.f;
    }
}
__global__ void k_set_steps(Scalars* sc, float a, float b, double* steps_out) {
    sc->step_a = a; sc->step_b = b;
    if (steps_out) { steps_out[0] = a; steps_out[1] = b; }
}

// ePIE-minibatch (R8) in ONE pass over a canvas: x += alpha n / (d + delta max); zero n and d.  which = 0: object (max = max_p2),
// 1: probe (max = max_dp).  (LSQML needs the directions before it knows its steps: k_direction, then k_apply.)
// The small per-batch jobs ride along instead of being launches of their own (config 1 is launch-bound: ten launches per batch
// became six).  which = 0 (object): the regulariser comes from sc->max_p2 (pi < 0) or sc->max_p2s[pi]; thread 0 zeroes sc->max_dp and
// sc->max_p2s[pw] for the kernels that follow (nobody reads them here).  which = 1 (probe): the step record is written, and with
// pw >= 0 the maximum of sum_k |P_k|^2 of the UPDATED probe is left in sc->max_p2s[pw] for the next batch.
__global__ void k_epie_update(float2* x, float2* n, float* d, size_t plane, int modes, float delta, float alpha, Scalars* sc, int which,
                              int update, int pi, int pw, double* steps_out, float step_a, float step_b) {
    const float reg = delta * (which ? sc->max_dp : (pi < 0 ? sc->max_p2 : sc->max_p2s[pi]));
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        if (!which) { sc->max_dp = 0.f; if (pw >= 0) sc->max_p2s[pw] = 0.f; }
        else if (steps_out) { steps_out[0] = step_a; steps_out[1] = step_b; }
    }
    float pm = 0.f;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < plane; i += (size_t)gridDim.x * blockDim.x) {
        const float st = alpha / (d[i] + reg);
        float p2 = 0.f;
        for (int k = 0; k < modes; ++k) {
            const size_t q = (size_t)k * plane + i;
            if (update || (which && pw >= 0)) {
                float2 xv = x[q];
                if (update) { const float2 nv = n[q]; xv.x = fmaf(st, nv.x, xv.x); xv.y = fmaf(st, nv.y, xv.y); x[q] = xv; }
                p2 = fmaf(xv.x, xv.x, fmaf(xv.y, xv.y, p2));
            }
            n[q] = make_float2(0.f, 0.f);
        }
        pm = fmaxf(pm, p2);
        d[i] = 0.f;
    }
    if (which && pw >= 0) {
        for (int s = 16; s > 0; s >>= 1) pm = fmaxf(pm, __shfl_xor_sync(0xffffffffu, pm, s));
        if ((threadIdx.x & 31) == 0) atomicMax(reinterpret_cast<unsigned int*>(&sc->max_p2s[pw]), __float_as_uint(pm));
    }
}

// x += step * dir; zero dir and d.  which = 0: step_a, 1: step_b.
__global__ void k_apply(float2* x, float2* dir, float* d, size_t plane, int modes, const Scalars* sc, int which,
                        int update) {
    const float st = which ? sc->step_b : sc->step_a;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < plane; i += (size_t)gridDim.x * blockDim.x) {
        for (int k = 0; k < modes; ++k) {
            const size_t q = (size_t)k * plane + i;
            if (update) { const float2 dv = dir[q]; float2 xv = x[q]; xv.x = fmaf(st, dv.x, xv.x); xv.y = fmaf(st, dv.y, xv.y); x[q] = xv; }
            dir[q] = make_float2(0.f, 0.f);
        }
        d[i] = 0.f;
    }
}

// sum of unmasked intensities in double (init).  part[block]; then k_finish_sum.
__global__ void k_sum_intensity(const void* __restrict__ I, int itype, size_t count, double* part) {
    double acc = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (size_t)gridDim.x * blockDim.x) {
        const float v = load_intensity(I, itype, i);
        if (v >= 0.f) acc += (double)v;
    }
    __shared__ double sa[32];
    for (int s = 16; s > 0; s >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, s);
    if ((threadIdx.x & 31) == 0) sa[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) { for (int w = 1; w < (int)blockDim.x / 32; ++w) acc += sa[w]; part[blockIdx.x] = acc; }
}
__global__ void k_finish_sum_I(const double* part, int n, Scalars* sc, int accumulate) {   // one warp, fixed order
    double s = 0;
    for (int i = threadIdx.x; i < n; i += 32) s += part[i];
    for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    if (threadIdx.x == 0) sc->sum_I = accumulate ? sc->sum_I + s : s;
}
__global__ void k_snap_sum_I(Scalars* sc) { sc->sum_I_iter = sc->sum_I; }
// E_t = (sum of all error partials, fixed order, double) / sum_I.  Two steps, both in a fixed order: kErrBlocks CTAs each
// reduce a contiguous piece to part[block]; the last CTA to finish (atomic ticket) adds the pieces in index order.
constexpr int kErrBlocks = 148;
__global__ void __launch_bounds__(1024) k_sum_error(const float* __restrict__ e_part, size_t count, const Scalars* sc, double* out, double* part,
                                                    unsigned int* ticket) {
    __shared__ double sa[32];
    __shared__ bool last;
    const size_t per = (count + gridDim.x - 1) / gridDim.x, i0 = blockIdx.x * per, i1 = min(count, i0 + per);
    double acc = 0.0;
    for (size_t i = i0 + threadIdx.x; i < i1; i += blockDim.x) acc += (double)e_part[i];
    for (int s = 16; s > 0; s >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, s);
    if ((threadIdx.x & 31) == 0) sa[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)blockDim.x / 32; ++w) acc += sa[w];
        part[blockIdx.x] = acc;
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last || threadIdx.x) return;
    __threadfence();
    double tot = 0.0;
    for (unsigned b = 0; b < gridDim.x; ++b) tot += __ldcg(part + b);
    *out = tot / (sc->sum_I_iter > 0 ? sc->sum_I_iter : 1.0);
    *ticket = 0;
}
__global__ void k_finish_init(Scalars* sc, float delta, int J, int which) {
    if (threadIdx.x || blockIdx.x) return;
    if (which == 0) sc->eps_O = delta * sc->max_p2;
    else { sc->eps_P = delta * (float)J * __uint_as_float(sc->max_bits); }
}

// ------------------------------------------------------------------------------------------
// probe-mode orthogonalisation (include/ptycho_b200.h: ptycho_orthogonalize_modes; reading R26)
// ------------------------------------------------------------------------------------------
// Gram matrix partials: grid (K*K, kGramBlocks); block (i*K + j, b) sums P_i conj(P_j) over its share of the pixels, in double.
constexpr int kGramBlocks = 32;
__global__ void __launch_bounds__(256) k_gram(const float2* __restrict__ P, int K, int nn, double2* __restrict__ part) {
    const int i = blockIdx.x / K, j = blockIdx.x % K;
    double re = 0.0, im = 0.0;
    for (int q = blockIdx.y * 256 + threadIdx.x; q < nn; q += gridDim.y * 256) {
        const float2 a = P[(size_t)i * nn + q], b = P[(size_t)j * nn + q];
        re += (double)a.x * b.x + (double)a.y * b.y;                  // a conj(b)
        im += (double)a.y * b.x - (double)a.x * b.y;
    }
    __shared__ double sr[8], si[8];
    for (int s = 16; s > 0; s >>= 1) { re += __shfl_xor_sync(0xffffffffu, re, s); im += __shfl_xor_sync(0xffffffffu, im, s); }
    if ((threadIdx.x & 31) == 0) { sr[threadIdx.x >> 5] = re; si[threadIdx.x >> 5] = im; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { re += sr[w]; im += si[w]; }
        part[blockIdx.x * gridDim.y + blockIdx.y] = make_double2(re, im);
    }
}
struct MixMatrix { float2 u[8][8]; };   // PTYCHO_MAX_MODES = 8
// x'_m = sum_k U[m][k] x_k at every pixel of every frame (in place).  grid (ceil(nn / 256), frames)
__global__ void __launch_bounds__(256) k_mix_modes(float2* __restrict__ x, int K, int nn, MixMatrix U) {
    const int q = blockIdx.x * 256 + threadIdx.x;
    if (q >= nn) return;
    float2* base = x + (size_t)blockIdx.y * K * nn + q;
    float2 in[8];
    for (int k = 0; k < K; ++k) in[k] = base[(size_t)k * nn];
    for (int m = 0; m < K; ++m) {
        float2 acc = make_float2(0.f, 0.f);
        for (int k = 0; k < K; ++k) acc = cadd(acc, cmul(U.u[m][k], in[k]));
        base[(size_t)m * nn] = acc;
    }
}

// ------------------------------------------------------------------------------------------
// init-time preparation of raw detector frames (include/ptycho_b200.h: ptycho_prepare_frames)
// ------------------------------------------------------------------------------------------
// (uy, ux) = source offset from the centre pixel for the output offset (dy, dx) after `rot` quarter turns counter-clockwise
// (R23; numpy.rot90 convention).
__device__ __forceinline__ void rot_offset(int rot, int dy, int dx, int& uy, int& ux) {
    switch (rot & 3) {
        case 0: uy = dy; ux = dx; break;
        case 1: uy = dx; ux = -dy; break;
        case 2: uy = -dy; ux = -dx; break;
        default: uy = -dx; ux = dy; break;
    }
}
template <typename TI, typename TO> __device__ __forceinline__ TO prepare_pixel(const TI* __restrict__ raw, size_t f, int det_h, int det_w, int sy,
                                                                                 int sx, float threshold, float saturation, float scale) {
    bool masked = sy < 0 || sx < 0 || sy >= det_h || sx >= det_w;
    float v = 0.f;
    if (!masked) {
        v = (float)__ldg(raw + (f * det_h + sy) * det_w + sx);
        if (sizeof(TI) == 2 && v == 65535.f) masked = true;            // already the sentinel
        if (sizeof(TI) == 4 && v < 0.f) masked = true;
        if (saturation > 0.f && v >= saturation) masked = true;
        if (threshold > 0.f && v < threshold) v = 0.f;
        v *= scale;                                                    // R24: per-frame normalisation, after the threshold
    }
    if (sizeof(TO) == 2) return (TO)(masked ? 65535.f : fminf(rintf(v), 65534.f));
    return (TO)(masked ? -1.0f : v);
}
// V output pixels along kx per thread (V = 8 when n % 16 == 0, no rotation and `out` is 16-byte aligned: one or two 16-byte
// stores; the V source pixels are contiguous too, because a group of 8 never straddles kx = n/2), else V = 1.
template <typename TI, typename TO, int V> __global__ void __launch_bounds__(256) k_prepare_frames(
    const TI* __restrict__ raw, int det_h, int det_w, int cy, int cx, int n, float threshold, float saturation, int rot,
    const float* __restrict__ frame_scale, TO* __restrict__ out, size_t total) {
    for (size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x; g * V < total; g += (size_t)gridDim.x * blockDim.x) {
        const size_t i = g * V;
        const int kx = (int)(i % n), ky = (int)((i / n) % n);
        const size_t f = i / ((size_t)n * n);
        const int dy = ky < n / 2 ? ky : ky - n, dx = kx < n / 2 ? kx : kx - n;
        const float sc = frame_scale ? __ldg(frame_scale + f) : 1.0f;
        TO v[V];
#pragma unroll
        for (int k = 0; k < V; ++k) {
            int uy, ux;
            rot_offset(rot, dy, dx + k, uy, ux);
            v[k] = prepare_pixel<TI, TO>(raw, f, det_h, det_w, cy + uy, cx + ux, threshold, saturation, sc);
        }
        if (V == 1) out[i] = v[0];
        else {
            const uint4* src = reinterpret_cast<const uint4*>(v);
#pragma unroll
            for (int k = 0; k < (int)(V * sizeof(TO) / 16); ++k) reinterpret_cast<uint4*>(out + i)[k] = src[k];
        }
    }
}

// ---- sub-pixel positions (reading R28) ---------------------------------------------------------------------
// ramp_d(k) = exp(-2 pi i (k_y d_y + k_x d_x) / N), k signed (k >= N/2 -> k - N).  Phase reduced in double: the argument reaches
// pi N and fp32 would lose the last digits of the fraction there.
__device__ __forceinline__ float2 shift_ramp(int ky, int kx, int n, float dy, float dx) {
    const int sy = ky < n / 2 ? ky : ky - n, sx = kx < n / 2 ? kx : kx - n;
    const double ph = -2.0 * ((double)sy * (double)dy + (double)sx * (double)dx) / (double)n;   // in units of pi
    double sn, cs;
    sincospi(ph, &sn, &cs);
    return make_float2((float)cs, (float)sn);
}
// Pj[f][k] = FP[k] * ramp_{delta_f}: the spectra of the shifted probes of this launch's frames.  grid (nframes, K n^2 / 256)
__global__ void k_sub_ramp(float2* __restrict__ Pj, const float2* __restrict__ FP, const float* __restrict__ frac, const int* __restrict__ frames,
                           int K, int n, float scale) {
    const size_t nn = (size_t)n * n, i = (size_t)blockIdx.y * blockDim.x + threadIdx.x;
    if (i >= nn * K) return;
    const int f = frames[blockIdx.x];
    const size_t q = i % nn;
    const float2 v = cmul(FP[i], shift_ramp((int)(q / n), (int)(q % n), n, frac[2 * f], frac[2 * f + 1]));
    Pj[(size_t)blockIdx.x * K * nn + i] = make_float2(v.x * scale, v.y * scale);   // scale = 1/n^2 of the inverse transform that follows
}
// nPF[k] += sum_f conj(ramp_{delta_f}) G[f][k]: the back-shifted probe terms of this launch, summed in Fourier space in frame order
// (fixed order, no atomics).  grid K n^2 / 256
__global__ void k_sub_acc(float2* __restrict__ nPF, const float2* __restrict__ G, const float* __restrict__ frac, const int* __restrict__ frames,
                          int nframes, int K, int n) {
    const size_t nn = (size_t)n * n, i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nn * K) return;
    const size_t q = i % nn;
    const int ky = (int)(q / n), kx = (int)(q % n);
    float2 acc = nPF[i];
    for (int s = 0; s < nframes; ++s) {
        const int f = frames[s];
        acc = cadd(acc, cmulc(G[(size_t)s * K * nn + i], shift_ramp(ky, kx, n, frac[2 * f], frac[2 * f + 1])));   // G conj(ramp)
    }
    nPF[i] = acc;
}
// LSQML with sub-pixel positions: the two sums that have no canvas closed form, from their per-frame definitions.
//   A22 = sum_j sum_k || dP_jk O_j ||^2,   A12 = Re sum_j sum_k conj(P_jk dO_j) (dP_jk O_j),   dP_jk = S_delta_j[dP_k]
// Pj, dPj: this launch's per-frame probes and probe directions (nframes x K x n x n).  grid (nframes, parts); fixed order, double.
__global__ void k_lsq_cross_pj(const float2* __restrict__ O, const float2* __restrict__ dO, int W, const float2* __restrict__ Pj,
                               const float2* __restrict__ dPj, int K, int n, int log2n, const YX* __restrict__ pos, const int* __restrict__ frames,
                               double* partX, double* partA22) {
    const YX p0 = pos[frames[blockIdx.x]];
    const int nn = n * n, stride = gridDim.y * blockDim.x;
    const size_t base = (size_t)p0.y * W + p0.x, fr = (size_t)blockIdx.x * K * nn;
    double a12 = 0.0, a22 = 0.0;
    for (int q = blockIdx.y * blockDim.x + threadIdx.x; q < nn; q += stride) {
        const size_t i = base + (size_t)(q >> log2n) * W + (q & (n - 1));
        const float2 o = __ldg(O + i), d = __ldg(dO + i);
        for (int k = 0; k < K; ++k) {
            const float2 u = cmul(Pj[fr + (size_t)k * nn + q], d), v = cmul(dPj[fr + (size_t)k * nn + q], o);
            a22 += (double)(v.x * v.x + v.y * v.y);
            a12 += (double)(u.x * v.x + u.y * v.y);
        }
    }
    __shared__ double sa[32], sb[32];
    for (int s = 16; s > 0; s >>= 1) { a12 += __shfl_xor_sync(0xffffffffu, a12, s); a22 += __shfl_xor_sync(0xffffffffu, a22, s); }
    if ((threadIdx.x & 31) == 0) { sa[threadIdx.x >> 5] = a12; sb[threadIdx.x >> 5] = a22; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)blockDim.x / 32; ++w) { a12 += sa[w]; a22 += sb[w]; }
        partX[blockIdx.x * gridDim.y + blockIdx.y] = a12; partA22[blockIdx.x * gridDim.y + blockIdx.y] = a22;
    }
}
// psi_jk = P_jk O_j for the slots of one launch (R4 initial exit waves with per-frame probes).  grid (nslots, K n^2 / 256)
__global__ void k_init_psi_pj(float2* __restrict__ psi, const float2* __restrict__ O, int W, const float2* __restrict__ Pj, int K, int n,
                              const YX* __restrict__ pos, const int* __restrict__ frames) {
    const size_t nn = (size_t)n * n, i = (size_t)blockIdx.y * blockDim.x + threadIdx.x;
    if (i >= nn * K) return;
    const size_t q = i % nn;
    const YX p0 = pos[frames[blockIdx.x]];
    psi[(size_t)blockIdx.x * K * nn + i] = cmul(Pj[(size_t)blockIdx.x * K * nn + i], O[(size_t)(p0.y + (int)(q / n)) * W + p0.x + (int)(q % n)]);
}
// dst = src * s (element-wise)
__global__ void k_scale_to(float2* __restrict__ dst, const float2* __restrict__ src, size_t n, float s) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) dst[i] = make_float2(src[i].x * s, src[i].y * s);
}

}  // namespace ptycho
