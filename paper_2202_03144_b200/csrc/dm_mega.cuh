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

// Experiment switches (m.flags: 1 = no L2 prefetch, 4 = immediate signals) exist in debug builds only (-DPTYCHO_DEBUG).
#ifdef PTYCHO_DEBUG
#define MEGA_FLAG(m, bit) ((m).flags & (bit))
#else
#define MEGA_FLAG(m, bit) 0
#endif

struct MegaArgs {
    FrameArgs f;        // psi = slot 0 of the store; S = ring base; frames = slot -> caller frame; e_part [J][NCB]
    int J, M, D, R, nW;
    int update_probe;   // accumulate the lagged probe sums (a9) in pass 1
    int fresh;          // first DM iteration after init / a minibatch algorithm: psi_j = P O_j (R4) is formed here, not read
    int corr;           // object canvas holds only the correction sum_j keep_j conj(P) v_j; d_O is gathered by k_dm_blend_gather (dm_det.cuh)
    int det;            // deterministic mode: no floating-point atomics here (dm_det.cuh forms the overlap sums)
    int pf;             // slots ahead that the L2 prefetches reach (megakernel: M, the next wave; split kernels: the next chunk)
    int flags;          // experiment switches (debug builds only): 1 = no L2 prefetch, 4 = immediate signals
    const void* It;     // intensities re-tiled at init into pass-2 register order (k_tile_intensity)
    const YX* spos;     // [J] position of each SLOT (pos[frames[slot]], one load instead of two chained)
    int* head;          // queue head
    int* cnt1;          // [J] pass-1 blocks done per slot
    int* cnt2;          // [J] pass-2 blocks done
    int* cnt2a;         // [J] split mode: error-only column blocks done (pass 2a)
    int* stat;          // [0] frames inside the power bound in the PREVIOUS iteration, [1] running count of this one
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
// "Ring slot read" needs no release: pass 3 signals only that its LOADS of S[slot] have completed (they
// have, the butterflies consumed them); nothing it writes is read again inside this kernel.  A relaxed
// increment spares the MEMBAR that would wait for the 48 stores and atomics of the previous slot.
__device__ __forceinline__ void warp_signal_relaxed(int* cnt) {
    __syncwarp();
    if ((threadIdx.x & 31) == 0) asm volatile("red.relaxed.gpu.global.add.s32 [%0], 1;" ::"l"(cnt) : "memory");
}
// -DPTYCHO_STRICT_SYNC builds the formally clean variant: the poll is an acquire (ptxas adds CCTL.IVALL: slower, see above).  In
// deterministic mode both variants must give bit-identical results (tests/test_gpu_parity.py::test_strict_sync_build_is_bit_identical).
__device__ __forceinline__ int ld_poll_gpu(const int* p) {
#ifdef PTYCHO_STRICT_SYNC
    return ld_acquire_gpu(p);
#else
    return ld_relaxed_gpu(p);
#endif
}
__device__ __forceinline__ void warp_wait(const int* cnt, int target) {
    if ((threadIdx.x & 31) == 0) {
        while (ld_poll_gpu(cnt) < target) __nanosleep(64);
    }
    __syncwarp();
}
// 1 - rb of the relaxed projection (R6) of one frame from its error partials, summed in a fixed order.
template <int N> __device__ __forceinline__ float frame_keep(const FrameArgs& a, int slot) {
    if (!(a.pbound > 0.f)) return 1.f;
    float e = 0.f;
    for (int i = 0; i < Geo<N>::NCB; ++i) e += __ldcg(a.e_part + (size_t)slot * Geo<N>::NCB + i);
    e *= 1.0f / ((float)N * (float)N);
    return (e <= a.pbound) ? 0.f : 1.f - sqrtf(a.pbound / e);
}
// HBM -> L2 ahead of use (no register or shared-memory cost); bytes is a multiple of 16.
// The prefetched data (exit waves, intensities) is streamed: used once, so it enters L2 as evict-first and does not push the
// ring S out (the ring is what should stay resident).
__device__ __forceinline__ void l2_prefetch_bulk(const void* p, uint32_t bytes) {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    asm volatile("cp.async.bulk.prefetch.L2.global.L2::cache_hint [%0], %1, %2;" ::"l"(p), "r"(bytes), "l"(pol) : "memory");
}
__device__ __forceinline__ void l2_prefetch(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
// A signal is sent one slot LATE (after the next slot's butterflies): by then the stores it covers
// have landed and the release fence (MEMBAR.GPU) does not stall the warp (ncu: 1.8 warps per issue
// were sitting in that fence).
struct Deferred {
    int* cnt = nullptr;
    __device__ __forceinline__ void flush_warp() { if (cnt) { warp_signal(cnt); cnt = nullptr; } }
    __device__ __forceinline__ void flush_cta_after_barrier() {   // caller: a CTA barrier has passed since the stores
        if (cnt) { if (threadIdx.x == 0) asm volatile("red.release.gpu.global.add.s32 [%0], 1;" ::"l"(cnt) : "memory"); cnt = nullptr; }
    }
};
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
#ifndef PTYCHO_MEGA_OCC
#define PTYCHO_MEGA_OCC 2      // resident CTAs per SM the register budget is sized for (N < 512)
#endif
constexpr int kWarps = kThreads / 32;

// Software phase profile (debug builds only, -DPTYCHO_PHASE_PROF): cycles per warp spent in each
// phase of each pass, summed over lane 0 of every warp.  [pass 0..2][wait, load, compute, store] + [12] = item fetch
#ifdef PTYCHO_PHASE_PROF
__device__ unsigned long long g_phase[16];
__shared__ unsigned long long s_phase[16];     // per CTA; flushed to g_phase when the kernel ends
struct PhaseClock {
    long long t; int base;
    __device__ __forceinline__ void start(int pass) { base = 4 * pass; t = clock64(); }
    __device__ __forceinline__ void lap(int phase) {
        const long long n = clock64();
        if ((threadIdx.x & 31) == 0) atomicAdd(&s_phase[base + phase], (unsigned long long)(n - t));
        t = n;
    }
};
#define PHASE_TOUCH(x) do { if ((x) == 1.2345e-33f) atomicAdd(&g_phase[15], 1ull); } while (0)
#else
struct PhaseClock {
    __device__ __forceinline__ void start(int) {}
    __device__ __forceinline__ void lap(int) {}
};
#define PHASE_TOUCH(x) do { } while (0)
#endif

// Init-time re-tiling of the intensities for pass 2 (run once).  The caller's
// row-major frames make a column block a 32-byte piece every 2 N bytes of DRAM (measured: those
// loads alone cost 3 ms of a 12 ms iteration); here the N x LPB block of (slot, blk) becomes one
// contiguous piece, ordered so that thread tid of pass 2 reads its E values as 16-byte chunks:
//   element (tid, r)  ->  chunk (r / EPC) * kThreads + tid, position r % EPC     (EPC = 16 / sizeof(T_I))
// with value I[frames[slot]][row = freq_b(t, r)][col = blk * LPB + c], c = tid % LPB, t = tid / LPB.
template <int N, typename TI> __global__ void __launch_bounds__(kThreads) k_tile_intensity(TI* __restrict__ out, const TI* __restrict__ I,
                                                                                            const int* __restrict__ frames) {
    using G = Geo<N>;
    constexpr int E = G::E, CB = G::LPB, EPC = 16 / (int)sizeof(TI);
    const int slot = blockIdx.x, blk = blockIdx.y, tid = threadIdx.x;
    const int c = tid % CB, t = tid / CB;
    const TI* src = I + (size_t)frames[slot] * N * N + blk * CB + c;
    TI* dst = out + ((size_t)slot * G::NCB + blk) * N * CB;
#pragma unroll
    for (int r = 0; r < E; ++r) dst[((size_t)(r / EPC) * kThreads + tid) * EPC + r % EPC] = src[(size_t)freq_b<N>(t, r) * N];
}

// The same re-tiling for a chunk of appended frames (streaming ingestion): frame `first + blockIdx.x` of the caller's numbering,
// read from the staged chunk, written to its slot.
template <int N, typename TI> __global__ void __launch_bounds__(kThreads) k_tile_intensity_chunk(TI* __restrict__ out, const TI* __restrict__ chunk,
                                                                                                  const int* __restrict__ slot_of, int first) {
    using G = Geo<N>;
    constexpr int E = G::E, CB = G::LPB, EPC = 16 / (int)sizeof(TI);
    const int slot = slot_of[first + blockIdx.x], blk = blockIdx.y, tid = threadIdx.x;
    const int c = tid % CB, t = tid / CB;
    const TI* src = chunk + (size_t)blockIdx.x * N * N + blk * CB + c;
    TI* dst = out + ((size_t)slot * G::NCB + blk) * N * CB;
#pragma unroll
    for (int r = 0; r < E; ++r) dst[((size_t)(r / EPC) * kThreads + tid) * EPC + r % EPC] = src[(size_t)freq_b<N>(t, r) * N];
}

template <int N> struct MegaGeo {
    using G = Geo<N>;
    static constexpr int LINE = (G::LS_ROW > G::LS_COL ? G::LS_ROW : G::LS_COL);
    static constexpr size_t smem = (size_t)(G::LPB * LINE + 2 * N * kTwWords + G::LPB * N) * sizeof(float2);   // exchange, twiddles, probe rows
};

// ---- pass 1: a1 exit wave, a2 reflector, a9 lagged probe sums, a3 forward row FFTs -> S --------
template <int N, bool SYNC = true> __device__ __forceinline__ void mega_pass1(const MegaArgs& m, int blk, int wave, float2* sm, const tw_t* s_tw,
                                                            Deferred& df, bool split) {
    using G = Geo<N>;
    constexpr int E = G::E, T = G::T, LW = 32 / T;
    const FrameArgs& a = m.f;
    const int l = threadIdx.x / T, t = threadIdx.x % T, lane = threadIdx.x & 31;
    float2* sx = sm + l * G::LS_ROW;
    const int y = blk * G::LPB + l;
    const size_t off = (size_t)y * N;
    float2 accN[E];                                                         // lagged probe sums of the M slots (R4)
    float accD[E];
#pragma unroll
    for (int i = 0; i < E; ++i) { accN[i] = make_float2(0.f, 0.f); accD[i] = 0.f; }
    const int s_begin = wave * m.M, s_end = min(m.J, (wave + 1) * m.M);
    float2* sP = reinterpret_cast<float2*>(const_cast<tw_t*>(s_tw) + 2 * N) + l * N;   // this line's probe row, kept for the M slots
#pragma unroll
    for (int i = 0; i < E; ++i) sP[t + T * i] = __ldg(a.P + off + t + T * i);
    __syncwarp();
    {   // psi of the NEXT wave's slots (this warp's lines): start HBM -> L2 now
        const int s = s_begin + m.pf + lane;
        if (!MEGA_FLAG(m, 1) && lane < m.M && s < m.J)
            l2_prefetch_bulk(a.psi + (size_t)s * N * N + (size_t)(blk * G::LPB + (threadIdx.x >> 5) * LW) * N, LW * N * 8);
    }
    PhaseClock pc;
    for (int slot = s_begin; slot < s_end; ++slot) {
        pc.start(0);
        if (SYNC && slot >= m.R) warp_wait(m.cnt3 + slot - m.R, G::NCB * kWarps);    // ring slot free again
        pc.lap(0);
        const YX p0 = m.spos[slot];
        const float2* orow = a.O + (size_t)(p0.y + y) * a.W + p0.x;
        const float2* prow = a.psi + (size_t)slot * N * N + off;
        float2 v[E];
#pragma unroll
        for (int i = 0; i < E; ++i) v[i] = m.fresh ? make_float2(0.f, 0.f) : __ldcs(prow + t + T * i);   // psi_j: streamed once
        float2 ov[E];
#pragma unroll
        for (int i = 0; i < E; ++i) ov[i] = __ldg(orow + t + T * i);
        df.flush_warp();                        // previous slot's signal: its fence waits while these loads are in flight anyway
        PHASE_TOUCH(v[E - 1].x);
        pc.lap(1);
#pragma unroll
        for (int i = 0; i < E; ++i) {
            const float2 o = ov[i];
            const float2 po = cmul(sP[t + T * i], o);                     // psi_O = P O_j
            const float2 s = m.fresh ? po : v[i];                         // R4: the initial exit wave is P O_j
            if (m.update_probe) {
                accN[i] = cadd(accN[i], cmulc(s, o));                     // conj(O_j) psi_j (lagged, R4)
                accD[i] = fmaf(o.x, o.x, fmaf(o.y, o.y, accD[i]));
            }
            v[i] = make_float2(fmaf(2.f, po.x, -s.x), fmaf(2.f, po.y, -s.y));   // reflector
            // split form: psi_j is overwritten with P O_j right away -- that IS the new exit wave of a frame inside its power bound
            // (keep = 0), so such a frame needs no pass 3 at all; a frame outside it has psi' = P O_j + keep v written by pass 3.
            if (split) __stcs(const_cast<float2*>(prow) + t + T * i, po);
        }
        fft_line_fwd<N, true>(v, t, sx, s_tw);
        __syncwarp();                                                       // sx is free for the next slot
        pc.lap(2);
        float2* srow = a.S + (size_t)(slot % m.R) * N * N + off;
#pragma unroll
        for (int r = 0; r < E; ++r) __stcg(srow + freq_b<N>(t, r), v[r]);
        if (SYNC) df.cnt = m.cnt1 + slot;
        if (MEGA_FLAG(m, 4)) df.flush_warp();
        pc.lap(3);
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
// MODE 0: the whole pass (fused form).  Split form, used when most frames were inside the power bound in the previous iteration (R6:
// their projection is the identity, so nothing has to be transformed back): MODE 1 = pass 2a, column FFTs and error partials only,
// S is left untouched; MODE 2 = the whole pass once more for ONE frame whose error turned out to exceed the bound (mega_pass2b
// below: pass 1 is known to be complete, no wait).  s_lo / s_hi >= 0 restrict the call to those slots of the wave.
enum { P2_FUSED = 0, P2_ERR_ONLY = 1, P2_REDO = 2 };
template <int N, bool U16, int MODE> __device__ __forceinline__ void mega_pass2(const MegaArgs& m, int blk, int wave, float2* sm, const tw_t* s_tw,
                                                            float* s_red, Deferred& df, int s_lo = -1, int s_hi = -1) {
    using G = Geo<N>;
    constexpr int E = G::E, T = G::T, CB = G::LPB;
    const FrameArgs& a = m.f;
    const int c = threadIdx.x % CB, t = threadIdx.x / CB;
    float2* sx = sm + c * G::LS_COL;
    const int col = blk * CB + c;
    constexpr float inv_n2 = 1.0f / ((float)N * (float)N);
    constexpr float kAmp2Floor = 1e-30f;
    const int s_begin = s_lo >= 0 ? s_lo : wave * m.M, s_end = s_lo >= 0 ? s_hi : min(m.J, (wave + 1) * m.M);
    const size_t tile_bytes = (size_t)N * CB * (U16 ? 2 : 4);   // this block's intensities of one slot: contiguous
    if (MODE != P2_REDO && !MEGA_FLAG(m, 1) && threadIdx.x < m.M) {           // I of the NEXT wave: HBM -> L2 now
        const int s = s_begin + m.pf + threadIdx.x;
        if (s < m.J) l2_prefetch_bulk(reinterpret_cast<const char*>(m.It) + ((size_t)s * G::NCB + blk) * tile_bytes, (uint32_t)tile_bytes);
    }
    PhaseClock pc;
    for (int slot = s_begin; slot < s_end; ++slot) {
        pc.start(1);
        if (MODE != P2_REDO) warp_wait(m.cnt1 + slot, G::NCB * kWarps);
        pc.lap(0);
        float2* base = a.S + (size_t)(slot % m.R) * N * N + col;
        float2 v[E];
#pragma unroll
        for (int i = 0; i < E; ++i) v[i] = __ldcg(base + (size_t)(t + T * i) * N);
        // I_j: streamed once as 16-byte chunks, kept packed in registers until the projection
        constexpr int NQ = U16 ? E / 8 : E / 4;
        uint4 iq[NQ];
        {
            const uint4* it = reinterpret_cast<const uint4*>(reinterpret_cast<const char*>(m.It) + ((size_t)slot * G::NCB + blk) * tile_bytes) + threadIdx.x;
#pragma unroll
            for (int j = 0; j < NQ; ++j) iq[j] = __ldcs(it + j * kThreads);
        }
        df.flush_cta_after_barrier();           // previous slot's signal: its fence waits while these loads are in flight anyway
        PHASE_TOUCH(v[E - 1].x + __uint_as_float(iq[NQ - 1].w));
        pc.lap(1);
        fft_line_fwd<N>(v, t, sx, s_tw);                                    // (CTA barrier inside)
        float err = 0.f;
#pragma unroll
        for (int r = 0; r < E; ++r) {
            const float a2 = fmaf(v[r].x, v[r].x, v[r].y * v[r].y);
            const bool pos = a2 > kAmp2Floor;                               // R2: below this |Phi| counts as 0
            const float ra = pos ? rsqrt_fast(a2) : 0.f;
            const float amp = a2 * ra;
            float inr;                                                      // R3: 65535 (u16) or a negative value = masked
            if (U16) {
                const unsigned w = (&iq[r / 8].x)[(r % 8) / 2];
                const unsigned u = (r & 1) ? (w >> 16) : (w & 0xffffu);
                inr = u == 65535u ? -1.0f : (float)u;
            } else inr = __uint_as_float((&iq[r / 4].x)[r % 4]);
            if (inr >= 0.f) {
                const float sq = sqrt_fast(inr), d = sq - amp;
                err = fmaf(d, d, err);
                if (pos) { const float sc = d * ra * inv_n2; v[r].x *= sc; v[r].y *= sc; }          // (s - 1)/N^2
                else v[r] = make_float2(sq * inv_n2, 0.f);                  // R2: Phi' - Phi = sqrt(I)
            } else v[r] = make_float2(0.f, 0.f);                            // R3: masked, Phi' - Phi = 0
        }
#pragma unroll
        for (int s = 16; s > 0; s >>= 1) err += __shfl_xor_sync(0xffffffffu, err, s);
        if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = err;
        __syncthreads();                                                    // sx free again; s_red visible
        if (MODE != P2_ERR_ONLY) fft_line_inv<N>(v, t, sx, s_tw + N);
        if (threadIdx.x == 0) {
            float tot = 0.f;
            for (int w = 0; w < kThreads / 32; ++w) tot += s_red[w];        // fixed order
            a.e_part[(size_t)slot * G::NCB + blk] = tot;
        }
        pc.lap(2);
        if (MODE == P2_ERR_ONLY) {
            __syncthreads();                                                // s_red free; e_part written
            df.cnt = m.cnt2a + slot;
            continue;
        }
#pragma unroll
        for (int r = 0; r < E; ++r) __stcg(base + (size_t)pos_a_inv<N>(t, r) * N, v[r]);
        __syncthreads();                                                    // sx and s_red free; stores issued by all
        df.cnt = m.cnt2 + slot;
        if (MEGA_FLAG(m, 4)) df.flush_cta_after_barrier();
        pc.lap(3);
    }
}

// ---- pass 2b of the split form: ONE item per wave.  For every frame of the wave: once all its error partials are there, a frame
// inside its power bound is passed on to pass 3 at once (the common case: a few microseconds per wave); a frame outside it gets
// the whole pass 2, all NCB column blocks, from this CTA (rare once the split form is in use).
template <int N, bool U16> __device__ __forceinline__ void mega_pass2b(const MegaArgs& m, int wave, float2* sm, const tw_t* s_tw, float* s_red,
                                                                       Deferred& df) {
    using G = Geo<N>;
    const int s_begin = wave * m.M, s_end = min(m.J, (wave + 1) * m.M);
    for (int slot = s_begin; slot < s_end; ++slot) {
        warp_wait(m.cnt2a + slot, G::NCB);                                  // every error partial of the frame is there
        if (frame_keep<N>(m.f, slot) == 0.f) {
            // Inside the bound: pass 1 has already written psi' = P O_j, nothing is scattered, S[slot] is not needed any more.  The
            // frame is marked "nothing to do" for pass 3 (counter value 2 NCB) and its ring slot is released here.
            __syncthreads();
            df.flush_cta_after_barrier();
            if (threadIdx.x == 0) {
                asm volatile("red.relaxed.gpu.global.add.s32 [%0], %1;" ::"l"(m.cnt2 + slot), "r"(2 * G::NCB) : "memory");
                asm volatile("red.relaxed.gpu.global.add.s32 [%0], %1;" ::"l"(m.cnt3 + slot), "r"(G::NCB * kWarps) : "memory");
                atomicAdd(m.stat + 1, 1);                                   // statistic for the next iteration's form
            }
            continue;
        }
        for (int blk = 0; blk < G::NCB; ++blk) mega_pass2<N, U16, P2_REDO>(m, blk, wave, sm, s_tw, s_red, df, slot, slot + 1);
    }
}

// ---- pass 3: a6 inverse row FFTs, a7 exit-wave update, a8 object scatter-add ---------------------
template <int N, bool SYNC = true> __device__ __forceinline__ void mega_pass3(const MegaArgs& m, int blk, int wave, float2* sm, const tw_t* s_tw,
                                                            Deferred& df, bool split) {
    using G = Geo<N>;
    constexpr int E = G::E, T = G::T;
    const FrameArgs& a = m.f;
    const int l = threadIdx.x / T, t = threadIdx.x % T;
    float2* sx = sm + l * G::LS_ROW;
    const int y = blk * G::LPB + l;
    const size_t off = (size_t)y * N;
    const int s_begin = wave * m.M, s_end = min(m.J, (wave + 1) * m.M);
    if (split && SYNC) {
        // One look at the whole wave first: if pass 2b has already marked every frame "inside its bound, nothing to do" (the steady
        // state), the item ends here -- one L2 round trip instead of one hand-off per slot and a staging of probe rows nobody uses.
        bool all_done = true;
        for (int k = threadIdx.x & 31; k < s_end - s_begin; k += 32) all_done = all_done && ld_relaxed_gpu(m.cnt2 + s_begin + k) >= 2 * G::NCB;
        if (__all_sync(0xffffffffu, all_done)) return;
    }
    float2* sP = reinterpret_cast<float2*>(const_cast<tw_t*>(s_tw) + 2 * N) + l * N;                                      // this line's probe row, kept for the M slots
#pragma unroll
    for (int i = 0; i < E; ++i) sP[t + T * i] = __ldg(a.P + off + t + T * i);
    __syncwarp();
    PhaseClock pc;
    for (int slot = s_begin; slot < s_end; ++slot) {
        pc.start(2);
        const YX p0 = m.spos[slot];                                         // (independent of the hand-off: in flight during the poll)
        if (SYNC) warp_wait(m.cnt2 + slot, G::NCB);
        if (split) {                                                        // split form: pass 2b marks a frame inside its bound with 2 NCB:
            int done = 0;                                                   // psi' = P O_j is already in the store (pass 1), the ring slot released
            if ((threadIdx.x & 31) == 0) done = ld_relaxed_gpu(m.cnt2 + slot) >= 2 * G::NCB;
            if (__shfl_sync(0xffffffffu, done, 0)) continue;
        }
        pc.lap(0);
        const size_t obase = (size_t)(p0.y + y) * a.W + p0.x;
        float2 o[E];                                                        // O_j (natural order), needed by both branches: issued before
#pragma unroll                                                              // the blend weight's loads, one latency for both
        for (int i = 0; i < E; ++i) o[i] = __ldg(a.O + obase + t + T * i);
        const float keep = frame_keep<N>(a, slot);                          // 1 - rb  (R6)
        float2* prow = a.psi + (size_t)slot * N * N + off;
        if (m.corr && !split && blk == 0 && threadIdx.x == 0 && keep == 0.f) atomicAdd(m.stat + 1, 1);   // statistic for the next iteration's form
        if (m.corr && keep == 0.f) {
            // The frame's error is inside the power bound (R6: rb = 1): the relaxed projection is the identity, psi' = P O_j, and the
            // frame adds nothing to the object correction (dm_det.cuh k_dm_blend_gather).  S[slot] is not read, nothing is transformed.
            if (SYNC) warp_signal_relaxed(m.cnt3 + slot);
#pragma unroll
            for (int i = 0; i < E; ++i) {
                const int x = t + T * i;
                __stcs(prow + x, cmul(sP[x], o[i]));
            }
            continue;
        }
        const float2* srow = a.S + (size_t)(slot % m.R) * N * N + off;
        float2 v[E];
#pragma unroll
        for (int r = 0; r < E; ++r) v[r] = __ldcg(srow + freq_b<N>(t, r));
        PHASE_TOUCH(v[E - 1].x + keep);
        pc.lap(1);
        fft_line_inv<N, true>(v, t, sx, s_tw + N);                          // v = F^-1[(s-1) Phi]
        __syncwarp();                                                       // sx is free for the next slot
        pc.lap(2);
        if (SYNC) warp_signal_relaxed(m.cnt3 + slot);                       // S[slot] has been read: the ring slot may be refilled
#pragma unroll
        for (int r = 0; r < E; ++r) {
            const int x = pos_a_inv<N>(t, r);
            const float2 p = sP[x];
            const float2 po = cmul(p, o[brev<E>(r)]);                     // x = t + T brev(r)
            const float2 kv = make_float2(keep * v[r].x, keep * v[r].y);
            const float2 w = cadd(po, kv);                                  // a7
            __stcs(prow + x, w);
            if (!m.det) {
                if (m.corr) red_add(a.nO + obase + x, cmulc(kv, p));        // a8, correction term only: keep conj(P) v
                else {
                    red_add(a.nO + obase + x, cmulc(w, p));                 // a8 conj(P) psi_j
                    red_add(a.dO + obase + x, fmaf(p.x, p.x, p.y * p.y));
                }
            }
        }
        pc.lap(3);
    }
}

template <int N, bool U16> __global__ void __launch_bounds__(kThreads, (N >= 512 ? 1 : PTYCHO_MEGA_OCC)) k_dm_mega(MegaArgs m) {
    using G = Geo<N>;
    extern __shared__ __align__(16) float2 sm[];
    tw_t* s_tw = reinterpret_cast<tw_t*>(sm + G::LPB * MegaGeo<N>::LINE);
    __shared__ float s_red[kThreads / 32];
    __shared__ int s_item;
    load_tw(s_tw, m.f.tw, m.f.twi, N);
    // split form when most frames were inside the power bound last time (their projection is the identity)
    const bool split = m.corr && m.f.pbound > 0.f && 2 * m.stat[0] > m.J;
    // fused form: NCB pass-3, NCB pass-2, NCB pass-1 items per queue wave, lags 2D / D / 0.  split form: NCB pass-3 items, ONE
    // pass-2b item, NCB pass-2a items, NCB pass-1 items, lags 3D / 2D / D / 0.
    const int per_qw = 3 * G::NCB + (split ? 1 : 0);
    const int total = (m.nW + (split ? 3 : 2) * m.D) * per_qw;
    Deferred df;
    bool df_cta = false;                                      // the pending signal is a CTA-level one (pass 2)
#ifdef PTYCHO_PHASE_PROF
    if (threadIdx.x < 16) s_phase[threadIdx.x] = 0;
    __syncthreads();
#endif
    PhaseClock pcf;
    for (;;) {
        pcf.start(3);
        __syncthreads();
        if (threadIdx.x == 0) s_item = atomicAdd(m.head, 1);
        __syncthreads();
        pcf.lap(0);
        // the last slot's signal of the previous item: must go out before this item can block on a flag
        if (df_cta) df.flush_cta_after_barrier(); else df.flush_warp();
        const int q = s_item;
        if (q >= total) break;
        const int qw = q / per_qw, idx = q % per_qw;
        int kind, blk;                                           // 0 pass 3, 1 pass 2 (fused) / 2b (split), 2 pass 2a (split only), 3 pass 1
        if (idx < G::NCB) { kind = 0; blk = idx; }
        else if (!split) { kind = idx < 2 * G::NCB ? 1 : 3; blk = idx % G::NCB; }
        else if (idx == G::NCB) { kind = 1; blk = 0; }
        else { kind = idx <= 2 * G::NCB ? 2 : 3; blk = (idx - 1) % G::NCB; }
        const int lag = kind == 3 ? 0 : split ? (3 - kind) : (2 - kind);
        const int wave = qw - lag * m.D;
        if (wave < 0 || wave >= m.nW) continue;
        df_cta = kind == 1 || kind == 2;
        if (kind == 3) mega_pass1<N>(m, blk, wave, sm, s_tw, df, split);
        else if (kind == 0) mega_pass3<N>(m, blk, wave, sm, s_tw, df, split);
        else if (!split) mega_pass2<N, U16, P2_FUSED>(m, blk, wave, sm, s_tw, s_red, df);
        else if (kind == 2) mega_pass2<N, U16, P2_ERR_ONLY>(m, blk, wave, sm, s_tw, s_red, df);
        else mega_pass2b<N, U16>(m, wave, sm, s_tw, s_red, df);
    }
#ifdef PTYCHO_PHASE_PROF
    __syncthreads();
    if (threadIdx.x < 16) atomicAdd(&g_phase[threadIdx.x], s_phase[threadIdx.x]);
#endif
}

}  // namespace ptycho
