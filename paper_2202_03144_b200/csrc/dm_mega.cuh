// dm_mega.cuh -- one persistent kernel per DM iteration (single probe mode), sm_100a.
//
// SURVEY.md 8(a) steps a1-a9 for every frame in ONE launch.  The three passes of kernels.cuh
// (forward rows | columns + modulus projection | inverse rows + update + scatter) become three
// item types of a single in-order work queue; CTAs pull items with one atomicAdd and hand frames
// from pass to pass through per-slot counters (release/acquire at gpu scope).  The half-transformed
// frame lives in a small ring S that stays in the 126 MB L2, so HBM sees psi in, psi out and I only.
//
// Queue order (deadlock-free by construction: every item depends only on items EARLIER in the
// queue, and an item is only ever held by a running CTA):
//   queue wave qw = 0 .. nW + 2D - 1 holds, in this order,
//     NCB items "pass 3" of frame wave qw - 2D, NCB items "pass 2" of wave qw - D, NCB items "pass 1" of wave qw.
//   A frame wave is M consecutive slots (spatially sorted frames); an item = (pass, block, wave)
//   loops over the M slots, so that pass 1 keeps the lagged probe sums (reading R4) in registers
//   and issues one atomic flush per M frames, and the probe rows of pass 1 / 3 stay in L1.
//   Ring: slot s uses S[s mod R], R >= (2D + 1) M, which makes "pass 3 of slot s - R" precede
//   "pass 1 of slot s" in the queue.
//
// Exit-wave update without re-reading psi: with phi = 2 psi_O - psi and the
// relaxed projection pf = rb phi + (1 - rb) F^-1[s Phi] (R6),
//   psi_new = psi + pf - psi_O = psi_O + (1 - rb) F^-1[(s - 1) Phi],
// so pass 2 scales by (s - 1)/N^2 and pass 3 needs only P and O_j.
#pragma once
#include "kernels.cuh"

namespace ptycho {

struct MegaArgs {
    FrameArgs f;        // psi = slot 0 of the store; S = ring base; frames = slot -> caller frame; e_part [J][NCB]
    int J, M, D, R, nW;
    int update_probe;   // accumulate the lagged probe sums (a9) in pass 1
    int* head;          // queue head
    int* cnt1;          // [J] pass-1 blocks done per slot
    int* cnt2;          // [J] pass-2 blocks done
    int* cnt3;          // [J] pass-3 blocks done
};

__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// All threads' prior global writes happen-before a consumer that acquires the counter.
__device__ __forceinline__ void slot_signal(int* cnt) {
    __syncthreads();
    if (threadIdx.x == 0) asm volatile("red.release.gpu.global.add.s32 [%0], 1;" ::"l"(cnt) : "memory");
}
__device__ __forceinline__ void slot_wait(const int* cnt, int target) {
    if (threadIdx.x == 0) {
        while (ld_acquire_gpu(cnt) < target) __nanosleep(100);
    }
    __syncthreads();
}
// Warp-granular forms: the row passes keep every line inside one warp, so warps signal and wait on
// their own and drift apart in phase (one warp's loads overlap another warp's butterflies).
//
// No gpu-scope ACQUIRE is used on the consumer side on purpose: an acquire (and __threadfence) makes
// ptxas emit CCTL.IVALL, which throws away the whole L1 -- and with it the probe rows and object
// tiles that every slot re-reads (ncu: 2.8 % L1 hit rate, P and O served from L2 each time).  The
// consumer polls with a relaxed load and then reads the producer's data only through ld.global.cg
// (L2, the point of coherence); the producer orders its st.global.cg writes before the counter
// increment with the release.  The poll's result is a control dependency of every later load.
__device__ __forceinline__ int ld_relaxed_gpu(const int* p) {
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void warp_signal(int* cnt) {
    __syncwarp();
    if ((threadIdx.x & 31) == 0) asm volatile("red.release.gpu.global.add.s32 [%0], 1;" ::"l"(cnt) : "memory");
}
__device__ __forceinline__ void warp_wait(const int* cnt, int target) {
    if ((threadIdx.x & 31) == 0) {
        while (ld_relaxed_gpu(cnt) < target) __nanosleep(64);
    }
    __syncwarp();
}
__device__ __forceinline__ float rsqrt_fast(float x) {
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float sqrt_fast(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
constexpr int kWarps = kThreads / 32;

template <int N> struct MegaGeo {
    using G = Geo<N>;
    static constexpr int LINE = (G::LS_ROW > G::LS_COL ? G::LS_ROW : G::LS_COL);
    static constexpr size_t smem = (size_t)(G::LPB * LINE + 2 * N) * sizeof(float2);
};

// ---- pass 1: a1 exit wave, a2 reflector, a9 lagged probe sums, a3 forward row FFTs -> S --------
template <int N> __device__ __forceinline__ void mega_pass1(const MegaArgs& m, int blk, int wave, float2* sm, const float2* s_tw) {
    using G = Geo<N>;
    constexpr int E = G::E, T = G::T;
    const FrameArgs& a = m.f;
    const int l = threadIdx.x / T, t = threadIdx.x % T;
    float2* sx = sm + l * G::LS_ROW;
    const int y = blk * G::LPB + l;
    const size_t off = (size_t)y * N;
    float2 accN[E];
    float accD[E];
#pragma unroll
    for (int i = 0; i < E; ++i) { accN[i] = make_float2(0.f, 0.f); accD[i] = 0.f; }
    const int s_end = min(m.J, (wave + 1) * m.M);
    for (int slot = wave * m.M; slot < s_end; ++slot) {
        const YX p0 = a.pos[a.frames[slot]];
        const float2* orow = a.O + (size_t)(p0.y + y) * a.W + p0.x;
        const float2* prow = a.psi + (size_t)slot * N * N + off;
        float2 v[E];
#pragma unroll
        for (int i = 0; i < E; ++i) v[i] = __ldcs(prow + t + T * i);      // psi_j: streamed from HBM once
#pragma unroll
        for (int i = 0; i < E; ++i) {
            const float2 o = __ldg(orow + t + T * i);
            const float2 po = cmul(__ldg(a.P + off + t + T * i), o);      // psi_O = P O_j
            const float2 s = v[i];
            if (m.update_probe) {
                accN[i] = cadd(accN[i], cmulc(s, o));                     // conj(O_j) psi_j (lagged, R4)
                accD[i] = fmaf(o.x, o.x, fmaf(o.y, o.y, accD[i]));
            }
            v[i] = make_float2(fmaf(2.f, po.x, -s.x), fmaf(2.f, po.y, -s.y));   // reflector
        }
        fft_line_fwd<N, true>(v, t, sx, s_tw);
        if (slot >= m.R) warp_wait(m.cnt3 + slot - m.R, G::NCB * kWarps);  // ring slot free again
        float2* srow = a.S + (size_t)(slot % m.R) * N * N + off;
#pragma unroll
        for (int r = 0; r < E; ++r) __stcg(srow + freq_b<N>(t, r), v[r]);
        warp_signal(m.cnt1 + slot);
    }
    if (m.update_probe) {
#pragma unroll
        for (int i = 0; i < E; ++i) {
            red_add(a.nP + off + t + T * i, accN[i]);
            red_add(a.dP + off + t + T * i, accD[i]);
        }
    }
}

// ---- pass 2: a3 column FFTs, a4 error partial, a5 modulus projection (as s - 1), a6 inverse columns
template <int N> __device__ __forceinline__ void mega_pass2(const MegaArgs& m, int blk, int wave, float2* sm, const float2* s_tw,
                                                            float* s_red) {
    using G = Geo<N>;
    constexpr int E = G::E, T = G::T, CB = G::LPB;
    const FrameArgs& a = m.f;
    const int c = threadIdx.x % CB, t = threadIdx.x / CB;
    float2* sx = sm + c * G::LS_COL;
    const int col = blk * CB + c;
    constexpr float inv_n2 = 1.0f / ((float)N * (float)N);
    constexpr float kAmp2Floor = 1e-30f;
    const int s_end = min(m.J, (wave + 1) * m.M);
    for (int slot = wave * m.M; slot < s_end; ++slot) {
        float2* base = a.S + (size_t)(slot % m.R) * N * N + col;
        const size_t ibase = (size_t)a.frames[slot] * N * N + col;
        float in[E];
#pragma unroll
        for (int r = 0; r < E; ++r) {                                       // I_j: streamed from HBM once
            const size_t idx = ibase + (size_t)freq_b<N>(t, r) * N;
            if (a.itype == 1) {
                const unsigned short u = __ldcs(reinterpret_cast<const unsigned short*>(a.I) + idx);
                in[r] = u == 65535 ? -1.0f : (float)u;
            } else in[r] = __ldcs(reinterpret_cast<const float*>(a.I) + idx);
        }
        warp_wait(m.cnt1 + slot, G::NCB * kWarps);
        float2 v[E];
#pragma unroll
        for (int i = 0; i < E; ++i) v[i] = __ldcg(base + (size_t)(t + T * i) * N);
        fft_line_fwd<N>(v, t, sx, s_tw);
        float err = 0.f;
#pragma unroll
        for (int r = 0; r < E; ++r) {
            const float a2 = fmaf(v[r].x, v[r].x, v[r].y * v[r].y);
            const bool pos = a2 > kAmp2Floor;                               // R2: below this |Phi| counts as 0
            const float ra = pos ? rsqrt_fast(a2) : 0.f;
            const float amp = a2 * ra;
            if (in[r] >= 0.f) {
                const float sq = sqrt_fast(in[r]), d = sq - amp;
                err = fmaf(d, d, err);
                if (pos) { const float sc = d * ra * inv_n2; v[r].x *= sc; v[r].y *= sc; }          // (s - 1)/N^2
                else v[r] = make_float2(sq * inv_n2, 0.f);                  // R2: Phi' - Phi = sqrt(I)
            } else v[r] = make_float2(0.f, 0.f);                            // R3: masked, Phi' - Phi = 0
        }
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) err += __shfl_xor_sync(0xffffffffu, err, s);
        if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = err;
        __syncthreads();                                                    // sx free again; s_red visible
        fft_line_inv<N>(v, t, sx, s_tw + N);
        if (threadIdx.x == 0) {
            float tot = 0.f;
            for (int w = 0; w < kThreads / 32; ++w) tot += s_red[w];        // fixed order
            a.e_part[(size_t)slot * G::NCB + blk] = tot;
        }
#pragma unroll
        for (int r = 0; r < E; ++r) __stcg(base + (size_t)pos_a_inv<N>(t, r) * N, v[r]);
        slot_signal(m.cnt2 + slot);
    }
}

// ---- pass 3: a6 inverse row FFTs, a7 exit-wave update, a8 object scatter-add ---------------------
template <int N> __device__ __forceinline__ void mega_pass3(const MegaArgs& m, int blk, int wave, float2* sm, const float2* s_tw) {
    using G = Geo<N>;
    constexpr int E = G::E, T = G::T;
    const FrameArgs& a = m.f;
    const int l = threadIdx.x / T, t = threadIdx.x % T;
    float2* sx = sm + l * G::LS_ROW;
    const int y = blk * G::LPB + l;
    const size_t off = (size_t)y * N;
    const int s_end = min(m.J, (wave + 1) * m.M);
    for (int slot = wave * m.M; slot < s_end; ++slot) {
        warp_wait(m.cnt2 + slot, G::NCB);
        float keep = 1.f;                                                   // 1 - rb  (R6)
        if (a.pbound > 0.f) {
            float e = 0.f;
            for (int i = 0; i < G::NCB; ++i) e += __ldcg(a.e_part + (size_t)slot * G::NCB + i);
            e *= 1.0f / ((float)N * (float)N);
            keep = (e <= a.pbound) ? 0.f : 1.f - sqrtf(a.pbound / e);
        }
        const YX p0 = a.pos[a.frames[slot]];
        const size_t obase = (size_t)(p0.y + y) * a.W + p0.x;
        const float2* srow = a.S + (size_t)(slot % m.R) * N * N + off;
        float2 v[E];
#pragma unroll
        for (int r = 0; r < E; ++r) v[r] = __ldcg(srow + freq_b<N>(t, r));
        fft_line_inv<N, true>(v, t, sx, s_tw + N);                          // v = F^-1[(s-1) Phi]
        float2* prow = a.psi + (size_t)slot * N * N + off;
#pragma unroll
        for (int r = 0; r < E; ++r) {
            const int x = pos_a_inv<N>(t, r);
            const float2 p = __ldg(a.P + off + x);
            const float2 po = cmul(p, __ldg(a.O + obase + x));
            const float2 w = make_float2(fmaf(keep, v[r].x, po.x), fmaf(keep, v[r].y, po.y));   // a7
            __stcs(prow + x, w);
            red_add(a.nO + obase + x, cmulc(w, p));                         // a8 conj(P) psi_j
            red_add(a.dO + obase + x, fmaf(p.x, p.x, p.y * p.y));
        }
        warp_signal(m.cnt3 + slot);
    }
}

template <int N> __global__ void __launch_bounds__(kThreads, (N >= 512 ? 1 : 2)) k_dm_mega(MegaArgs m) {
    using G = Geo<N>;
    extern __shared__ float2 sm[];
    float2* s_tw = sm + G::LPB * MegaGeo<N>::LINE;
    __shared__ float s_red[kThreads / 32];
    __shared__ int s_item;
    load_tw(s_tw, m.f.tw, m.f.twi, N);
    const int per_qw = 3 * G::NCB;
    const int total = (m.nW + 2 * m.D) * per_qw;
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_item = atomicAdd(m.head, 1);
        __syncthreads();
        const int q = s_item;
        if (q >= total) break;
        const int qw = q / per_qw, idx = q % per_qw;
        const int kind = idx / G::NCB, blk = idx % G::NCB;    // 0: pass 3, 1: pass 2, 2: pass 1
        const int wave = qw - (2 - kind) * m.D;
        if (wave < 0 || wave >= m.nW) continue;
        if (kind == 2) mega_pass1<N>(m, blk, wave, sm, s_tw);
        else if (kind == 1) mega_pass2<N>(m, blk, wave, sm, s_tw, s_red);
        else mega_pass3<N>(m, blk, wave, sm, s_tw);
    }
}

}  // namespace ptycho
