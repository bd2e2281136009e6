// The 256-point line FFT as two radix-16 stages on the tensor cores -- a MICRO-BENCHMARK, not part of the product path.
//
// BASELINE.json's north_star asks whether the DFT-as-GEMM route can beat the packed-fp32 line FFT at <= 2e-6 error; the round-1
// review asked for a time-boxed measurement rather than the paper argument of DESIGN.md section 7.  This is that measurement's
// kernel (entry point ptycho_test_fft_rows, impl = 1; bench.py --mma-dft times it beside the product's row pass).
//
// One warp transforms one line, entirely in registers -- no shared memory, which is the pipe that binds the product kernel:
//   n = 16 n1 + n2, k = k1 + 16 k2:   X[k] = sum_n2 W16^(n2 k2) * [ W256^(n2 k1) * sum_n1 W16^(n1 k1) x[16 n1 + n2] ]
//   stage 1   Y  = F16 . Xm           (16 x 16 complex;  A = F16 (constant fragments), B = Xm[n1][n2] loaded straight from global)
//   twiddle   Y' = Y o W256^(k1 n2)   (element-wise on the accumulator fragments; per-thread constants)
//   stage 2   Z  = Y' . F16           (A = Y': the accumulator fragment of stage 1 IS an A fragment of mma.m16n8k8 up to a
//                                      permutation of the contraction index, which is folded into the rows of the constant B = F16)
//   X[k1 + 16 k2] = Z[k1][k2]
// mma.sync.m16n8k8 TF32 with the 3-term split x = hi + lo (hi = tf32(x), lo = tf32(x - hi);  a b ~ a_lo b_hi + a_hi b_lo + a_hi b_hi),
// fp32 accumulation: 96 MMAs per line (2 stages x 4 real products x 4 tiles x 3 terms).  Fragment layouts (verified on the device
// against a plain matrix product): g = lane / 4, t = lane % 4;  A: (g, t) (g+8, t) (g, t+4) (g+8, t+4);  B: (k = t, n = g) (t+4, g);
// C: (g, 2t) (g, 2t+1) (g+8, 2t) (g+8, 2t+1).
#pragma once
#include <cuda_runtime.h>

namespace ptycho {

__device__ __forceinline__ unsigned to_tf32(float x) {
    unsigned r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ void split_tf32(float x, unsigned& hi, unsigned& lo) {
    hi = to_tf32(x);
    lo = to_tf32(x - __uint_as_float(hi));
}
__device__ __forceinline__ void mma_tf32(float (&c)[4], const unsigned (&a)[4], unsigned b0, unsigned b1) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// c += a b with both operands split in two: the small terms first
__device__ __forceinline__ void mma3(float (&c)[4], const unsigned (&ah)[4], const unsigned (&al)[4], const unsigned (&bh)[2], const unsigned (&bl)[2]) {
    mma_tf32(c, al, bh[0], bh[1]);
    mma_tf32(c, ah, bl[0], bl[1]);
    mma_tf32(c, ah, bh[0], bh[1]);
}
// exp(-2 pi i m / 16) in double (the constant DFT matrix is split into hi + lo like the data), and the stage twiddles in fp32
__constant__ double2 kW16[16] = {{1, -0}, {0.92387953251128674, -0.38268343236508978}, {0.70710678118654757, -0.70710678118654746}, {0.38268343236508984, -0.92387953251128674}, {6.123233995736766e-17, -1}, {-0.38268343236508973, -0.92387953251128674}, {-0.70710678118654746, -0.70710678118654757}, {-0.92387953251128674, -0.38268343236508989}, {-1, -1.2246467991473532e-16}, {-0.92387953251128685, 0.38268343236508967}, {-0.70710678118654768, 0.70710678118654746}, {-0.38268343236509034, 0.92387953251128652}, {-1.8369701987210297e-16, 1}, {0.38268343236509, 0.92387953251128663}, {0.70710678118654735, 0.70710678118654768}, {0.92387953251128652, 0.38268343236509039}};
__device__ __forceinline__ void split_tf32_d(double v, unsigned& hi, unsigned& lo) {
    hi = to_tf32((float)v);
    lo = to_tf32((float)(v - (double)__uint_as_float(hi)));
}
__device__ __forceinline__ float2 root256(int m) {                          // exp(-2 pi i m / 256)
    float s, c;
    sincospif(-(float)(m & 255) * (1.0f / 128.0f), &s, &c);
    return make_float2(c, s);
}

// data: nlines lines of 256 complex64, transformed in place (forward, unscaled, natural order in and out).
__global__ void __launch_bounds__(128, 4) k_rows_mma256(float2* __restrict__ data, long long nlines) {
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    // ---- per-thread constants --------------------------------------------------------------------------------------------
    unsigned Arh[2][4], Arl[2][4], Aih[2][4], Ail[2][4];                    // stage 1: A = F16[k1][n1], chunk c: n1 = 8c + {t, t+4}
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int row = g + 8 * (e & 1), col = 8 * c + t + 4 * (e >> 1);
            const double2 w = kW16[(row * col) & 15];
            split_tf32_d(w.x, Arh[c][e], Arl[c][e]);
            split_tf32_d(w.y, Aih[c][e], Ail[c][e]);
        }
    unsigned Brh[2][2][2], Brl[2][2][2], Bih[2][2][2], Bil[2][2][2];        // stage 2: B = F16[n2][k2]; chunk c: contraction slot t <-> n2 = 8c + 2t,
#pragma unroll                                                               // slot t+4 <-> n2 = 8c + 2t + 1 (the accumulator's columns); tile j: k2 = 8j + g
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const double2 w = kW16[((8 * c + 2 * t + e) * (8 * j + g)) & 15];
                split_tf32_d(w.x, Brh[c][j][e], Brl[c][j][e]);
                split_tf32_d(w.y, Bih[c][j][e], Bil[c][j][e]);
            }
    float2 tw[2][4];                                                        // W256^(k1 n2) at the accumulator's positions of tile j
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
        for (int e = 0; e < 4; ++e) tw[j][e] = root256((g + 8 * (e >> 1)) * (8 * j + 2 * t + (e & 1)));

    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long line = warp; line < nlines; line += nwarps) {
        float2* x = data + line * 256;
        // B operands of stage 1: Xm[n1][n2] = x[16 n1 + n2];  chunk c, tile j: (n1 = 8c + t, n2 = 8j + g), (n1 = 8c + t + 4, n2 = 8j + g)
        float2 xv[2][2][2];
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int j = 0; j < 2; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) xv[c][j][e] = x[16 * (8 * c + t + 4 * e) + 8 * j + g];
        float Yr[2][4], Yi[2][4];
#pragma unroll
        for (int j = 0; j < 2; ++j) {
#pragma unroll
            for (int e = 0; e < 4; ++e) { Yr[j][e] = 0.f; Yi[j][e] = 0.f; }
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                unsigned rh[2], rl[2], ih[2], il[2], nh[2], nl[2];
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    split_tf32(xv[c][j][e].x, rh[e], rl[e]);
                    split_tf32(xv[c][j][e].y, ih[e], il[e]);
                    nh[e] = ih[e] ^ 0x80000000u; nl[e] = il[e] ^ 0x80000000u;   // -Im x
                }
                mma3(Yr[j], Arh[c], Arl[c], rh, rl);                        // Re Y = Fr Xr - Fi Xi
                mma3(Yr[j], Aih[c], Ail[c], nh, nl);
                mma3(Yi[j], Arh[c], Arl[c], ih, il);                        // Im Y = Fr Xi + Fi Xr
                mma3(Yi[j], Aih[c], Ail[c], rh, rl);
            }
        }
        // twiddle, and the accumulator of tile j becomes the A operand of contraction chunk c = j: (c0, c2, c1, c3)
        unsigned Yrh[2][4], Yrl[2][4], Yih[2][4], Yil[2][4], Ynh[2][4], Ynl[2][4];
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const float yr = Yr[j][e] * tw[j][e].x - Yi[j][e] * tw[j][e].y, yi = Yr[j][e] * tw[j][e].y + Yi[j][e] * tw[j][e].x;
                const int a = (e == 1) ? 2 : (e == 2) ? 1 : e;
                split_tf32(yr, Yrh[j][a], Yrl[j][a]);
                split_tf32(yi, Yih[j][a], Yil[j][a]);
                Ynh[j][a] = Yih[j][a] ^ 0x80000000u; Ynl[j][a] = Yil[j][a] ^ 0x80000000u;
            }
#pragma unroll
        for (int j = 0; j < 2; ++j) {                                       // output tile j: k2 = 8j + {2t, 2t+1}
            float Zr[4] = {0.f, 0.f, 0.f, 0.f}, Zi[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                mma3(Zr, Yrh[c], Yrl[c], Brh[c][j], Brl[c][j]);             // Re Z = Y'r Fr - Y'i Fi
                mma3(Zr, Ynh[c], Ynl[c], Bih[c][j], Bil[c][j]);
                mma3(Zi, Yrh[c], Yrl[c], Bih[c][j], Bil[c][j]);             // Im Z = Y'r Fi + Y'i Fr
                mma3(Zi, Yih[c], Yil[c], Brh[c][j], Brl[c][j]);
            }
#pragma unroll
            for (int e = 0; e < 4; ++e) x[(g + 8 * (e >> 1)) + 16 * (8 * j + 2 * t + (e & 1))] = make_float2(Zr[e], Zi[e]);   // X[k1 + 16 k2]
        }
    }
}

}  // namespace ptycho
