// fft_core.cuh -- register-blocked two-stage complex64 FFT lines for N = 64..512 (sm_100a).
//
// Step a3/a6 of SURVEY.md 8(a) (north_star: "shared-memory batched radix-4/8 complex64 FFT for
// 64-512 sizes").  Differs from the north_star wording in one way, stated in DESIGN.md: each 1-D
// transform is TWO register-resident radix-E / radix-T passes (E*T = N, E in {8,16,32}) with a
// single shared-memory exchange between them, instead of log4(N) shared-memory radix-4 passes;
// SURVEY.md H1 asks for exactly this to stay under the shared-memory ceiling.
//
// A "line" of N points is owned by T threads.  Two register layouts:
//   layout A (space side):     thread b holds x[b + T*a],               a = 0..E-1
//   layout B (frequency side): thread t holds X[(t + T*m) + E*kb],      m < E/T, kb < T
// forward : A -> B,  X[k] = sum_n x[n] exp(-2 pi i n k / N)   (unnormalised, reading R1)
// inverse : B -> A,  x[n] = sum_k X[k] exp(+2 pi i n k / N)   (caller folds the 1/N)
#pragma once
#include <cuda_runtime.h>

namespace ptycho {

template <int N> struct FftCfg;
template <> struct FftCfg<64>  { static constexpr int E = 8,  T = 8;  };
template <> struct FftCfg<128> { static constexpr int E = 16, T = 8;  };
template <> struct FftCfg<256> { static constexpr int E = 16, T = 16; };
template <> struct FftCfg<512> { static constexpr int E = 32, T = 16; };

__host__ __device__ constexpr int ilog2c(int v) { return v <= 1 ? 0 : 1 + ilog2c(v >> 1); }
template <int R> __host__ __device__ constexpr int brev(int i) {
    int r = 0;
    for (int b = 0; b < ilog2c(R); ++b) r |= ((i >> b) & 1) << (ilog2c(R) - 1 - b);
    return r;
}

// Complex arithmetic on packed pairs.  sm_100a has two-wide fp32 instructions (FADD2 / FMUL2 / FFMA2,
// PTX add/mul/fma.f32x2) whose operands can swap and negate their halves for free, so a complex add,
// a rotation by +-i folded into an add, and each half of a complex multiply are ONE issue slot each.
// The fp32 pipe rate is the same as for scalar code (measured: 127 against 125 lane-ops/clk/SM); what
// halves is the number of instructions a warp has to issue, which is what bounds this kernel (ncu:
// 40 % issue-active at 16 warps per SM, "wait" and "short scoreboard" stalls).
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {   // a * b
    return __ffma2_rn(make_float2(a.y, a.x), make_float2(-b.y, b.y), __fmul2_rn(a, make_float2(b.x, b.x)));
}
__device__ __forceinline__ float2 cmulc(float2 a, float2 b) {  // a * conj(b)
    return __ffma2_rn(make_float2(a.y, a.x), make_float2(b.y, -b.y), __fmul2_rn(a, make_float2(b.x, b.x)));
}
// Twiddle tables hold w = (c, s) as the four words {c, c, -s, s}: y * w and y * conj(w) are then one
// FMUL2 and one FFMA2 with no register shuffling.
__device__ __forceinline__ float4 tw_pack(float2 w) { return make_float4(w.x, w.x, -w.y, w.y); }
// The twiddle tables sit in shared memory as plain float2 and are packed after the load: half the bytes through the shared-memory
// pipe, which is the one that binds (measured at config 2: 8.02 -> 7.90 ms per early iteration against float4 entries).
using tw_t = float2;
constexpr int kTwWords = sizeof(tw_t) / sizeof(float2);      // table entry size in float2 units (shared-memory sizing)

__device__ __forceinline__ float2 cmul_tw(float2 y, float4 w) {
    return __ffma2_rn(make_float2(y.y, y.x), make_float2(w.z, w.w), __fmul2_rn(y, make_float2(w.x, w.y)));
}
__device__ __forceinline__ float2 cmulc_tw(float2 y, float4 w) {
    return __ffma2_rn(make_float2(y.y, y.x), make_float2(-w.z, -w.w), __fmul2_rn(y, make_float2(w.x, w.y)));
}
__device__ __forceinline__ float2 cmul_tw(float2 y, float2 w) { return cmul_tw(y, tw_pack(w)); }
__device__ __forceinline__ float2 cmulc_tw(float2 y, float2 w) { return cmulc_tw(y, tw_pack(w)); }
__device__ __forceinline__ float4 tw_store(float2 w, float4*) { return tw_pack(w); }
__device__ __forceinline__ float2 tw_store(float2 w, float2*) { return w; }

// cos(2 pi m / 32), sin(2 pi m / 32): literals so that unrolled butterflies get immediates.
__device__ __forceinline__ constexpr float cos32(int m) {
    constexpr float c[9] = {1.0f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                            0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f,
                            0.19509032201612826785f, 0.0f};
    m &= 31;
    return m <= 8 ? c[m] : m <= 16 ? -c[16 - m] : m <= 24 ? -c[m - 16] : c[32 - m];
}
__device__ __forceinline__ constexpr float sin32(int m) { return cos32(m - 8); }

// d * exp(-+ 2 pi i m / R) with m known after unrolling; trivial factors cost no multiply.
template <int R, bool INV> __device__ __forceinline__ float2 mul_root(float2 d, int m) {
    constexpr float h = 0.70710678118654752440f;
    if (m == 0) return d;
    if (4 * m == R) return INV ? make_float2(-d.y, d.x) : make_float2(d.y, -d.x);       // folds into the next add
    if (8 * m == R)
        return __fmul2_rn(__fadd2_rn(d, INV ? make_float2(-d.y, d.x) : make_float2(d.y, -d.x)), make_float2(h, h));
    if (8 * m == 3 * R)
        return __fmul2_rn(__fadd2_rn(make_float2(-d.x, -d.y), INV ? make_float2(-d.y, d.x) : make_float2(d.y, -d.x)), make_float2(h, h));
    const float c = cos32(m * (32 / R)), s = sin32(m * (32 / R));
    return __ffma2_rn(make_float2(d.y, d.x), INV ? make_float2(-s, s) : make_float2(s, -s), __fmul2_rn(d, make_float2(c, c)));
}

// In-register R-point DFT (decimation in frequency).  In: v[n] natural.  Out: v[i] = Y[brev<R>(i)].
template <int R, bool INV> __device__ __forceinline__ void dft_reg(float2 (&v)[R]) {
#pragma unroll
    for (int half = R / 2; half >= 1; half >>= 1) {
#pragma unroll
        for (int blk = 0; blk < R; blk += 2 * half) {
#pragma unroll
            for (int j = 0; j < half; ++j) {
                const float2 a = v[blk + j], b = v[blk + j + half];
                v[blk + j] = cadd(a, b);
                v[blk + j + half] = mul_root<R, INV>(csub(a, b), j * (R / (2 * half)));
            }
        }
    }
}

// Shared-memory exchange region of one line: E rows of (T+1) float2 (padding keeps the
// transposed access conflict-free when lanes run along b); LS = line stride in float2.
template <int N> struct LineSmem {
    static constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T, LD = T + 1;
    static constexpr int SIZE = E * LD;
};

// layout-B bookkeeping: register r of thread t holds frequency index freq_b<N>(t, r).
template <int N> __device__ __forceinline__ constexpr int freq_b(int t, int r) {
    constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T;
    return t + T * (r / T) + E * brev<T>(r % T);
}
// layout-A bookkeeping after an inverse line: register r of thread b holds x[b + T*brev<E>(r)].
template <int N> __device__ __forceinline__ constexpr int pos_a_inv(int b, int r) {
    return b + FftCfg<N>::T * brev<FftCfg<N>::E>(r);
}

// Forward line, A -> B.  v[a] = x[t + T*a] on entry (natural a); v[r] = X[freq_b(t, r)] on exit.
// sx: this line's exchange region; tw[ka*T + b] = exp(-2 pi i b ka / N) (packed for the f32x2 multiply after the load).  All threads of the CTA
// must call (contains __syncthreads).
template <bool WARP> __device__ __forceinline__ void line_sync() {
    if (WARP) __syncwarp(); else __syncthreads();
}

// WARP = true: every line's T threads sit in one warp (row passes), so the exchange needs only a
// warp barrier and warps run independently of one another.
template <int N, bool WARP = false> __device__ __forceinline__ void fft_line_fwd(float2 (&v)[FftCfg<N>::E], int t, float2* sx,
                                                              const tw_t* __restrict__ tw) {
    constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T, LD = LineSmem<N>::LD;
    dft_reg<E, false>(v);
#pragma unroll
    for (int i = 0; i < E; ++i) {
        const int ka = brev<E>(i);
        float2 y = v[i];
        if (ka) y = cmul_tw(y, tw[ka * T + t]);
        sx[ka * LD + t] = y;
    }
    line_sync<WARP>();
#pragma unroll
    for (int m = 0; m < E / T; ++m) {
        float2 u[T];
#pragma unroll
        for (int b = 0; b < T; ++b) u[b] = sx[(t + T * m) * LD + b];
        dft_reg<T, false>(u);
#pragma unroll
        for (int i = 0; i < T; ++i) v[m * T + i] = u[i];
    }
}

// Inverse line, B -> A (unnormalised).  v[r] = X[freq_b(t, r)] on entry; v[r] = x[pos_a_inv(t, r)]
// on exit.  twi[b*E + ka] = exp(-2 pi i b ka / N) (same values as tw, transposed so that lanes,
// which run along ka here, read consecutive words).  Contains __syncthreads.
template <int N, bool WARP = false> __device__ __forceinline__ void fft_line_inv(float2 (&v)[FftCfg<N>::E], int t, float2* sx,
                                                              const tw_t* __restrict__ twi) {
    constexpr int E = FftCfg<N>::E, T = FftCfg<N>::T, LD = LineSmem<N>::LD;
#pragma unroll
    for (int m = 0; m < E / T; ++m) {
        float2 u[T];
#pragma unroll
        for (int kb = 0; kb < T; ++kb) u[kb] = v[m * T + brev<T>(kb)];
        dft_reg<T, true>(u);  // u[i] = Z[b = brev<T>(i)] for ka = t + T*m
        const int ka = t + T * m;
#pragma unroll
        for (int i = 0; i < T; ++i) {
            const int b = brev<T>(i);
            sx[ka * LD + b] = b ? cmulc_tw(u[i], twi[b * E + ka]) : u[i];
        }
    }
    line_sync<WARP>();
#pragma unroll
    for (int ka = 0; ka < E; ++ka) v[ka] = sx[ka * LD + t];
    dft_reg<E, true>(v);
}

}  // namespace ptycho
