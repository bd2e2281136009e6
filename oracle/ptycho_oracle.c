/* ptycho_oracle.c -- plain, slow CPU oracle for the ptychographic projection cycle.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call this file.  It shares
 * no code, table, header or helper with paper_2202_03144_b200/csrc (the CUDA path) and neither
 * imports the other.
 *
 * What it follows.  /root/reference/PAPER.md gives no equations (it is a software paper); the
 * cycle is the one stated in BASELINE.json `north_star` ("forms the exit wave psi_j = P * O[r_j]
 * ... 2-D FFT, replaces the Fourier modulus with sqrt(I_j) (DM additionally applies the
 * reflector ...) ... inverse FFT, then scatter-adds the overlap update of object and probe"),
 * PAPER.md:58 (DM keeps the previous exit waves and processes all scan points at once; ePIE has
 * the small footprint), PAPER.md:52 (probe update can start at a later iteration)
 * (several probe modes), and the step-by-step restatement in SURVEY.md section 8(c) (items C1-C3,
 * "DM", "ePIE-minibatch", "LSQML-style minibatch", readings R1-R9).  Each function cites its
 * item.  The method is an iteration, so the oracle is the algorithm step by step, in that order,
 * in double precision (build with -DORACLE_FLOAT for the fp32 drift-floor variant).
 *
 * Parity pins (tests/test_oracle_pins.py): FFT vs brute-force DFT, numpy's FFT, Parseval, delta
 * and plane-wave closed forms; projection: |Phi'|^2 = I, phase kept, idempotent, relaxed closed
 * form; zero error and fixed point at ground truth; closed-form overlap update; ePIE<->DM
 * cross-check; LSQML K=1 / forced steps <-> ePIE; step solve vs numpy.linalg.lstsq of the explicit
 * system; symmetries; eval_error off zero against numpy's FFT; the probe direction n_P/(d_P + delta max d_P) from numpy
 * slices; masked pixels excluded from sum I; the sequential overlap projection against the overlap closed forms; B = 1
 * against single-frame steps in sequence; the per-frame steps against per-frame numpy.linalg.lstsq and the weighted-scatter
 * formula.  PARITY UNPINNED: fidelity of "LSQML-style" (R9) and of its per-frame variant (R25) to the LSQML of the paper's
 * ref [18] (that text is not available; both readings are definitions, not reproductions).
 *
 * Parallelism: OpenMP over frames for the per-frame transforms only; every cross-frame sum is
 * accumulated serially in frame order, so results do not depend on the thread count.
 */
#define _GNU_SOURCE
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORACLE_FLOAT
typedef float real;
typedef float complex cplx;
#define CABS2(z) (crealf(z) * crealf(z) + cimagf(z) * cimagf(z))
#define SQRT sqrtf
#else
typedef double real;
typedef double complex cplx;
#define CABS2(z) (creal(z) * creal(z) + cimag(z) * cimag(z))
#define SQRT sqrt
#endif

#define ALG_EPIE_MB 0
#define ALG_DM 1
#define ALG_LSQML 2

int orc_real_bytes(void) { return (int)sizeof(real); }

/* ------------------------------------------------------------------------------------------
 * Fourier transforms (reading R1: F unnormalised forward, DC at [0,0]; F^-1 carries 1/N^2).
 * ------------------------------------------------------------------------------------------ */

/* Definition of the 2-D DFT written out, O(n^4).  Pins the fast transform below. */
void orc_dft2_naive(int n, const cplx *in, cplx *out, int inverse) {
    const double sgn = inverse ? 1.0 : -1.0;
    for (int u = 0; u < n; ++u)
        for (int v = 0; v < n; ++v) {
            double complex acc = 0;
            for (int y = 0; y < n; ++y)
                for (int x = 0; x < n; ++x) {
                    double ang = sgn * 2.0 * M_PI * ((double)u * y + (double)v * x) / n;
                    acc += (double complex)in[y * n + x] * (cos(ang) + I * sin(ang));
                }
            out[u * n + v] = (cplx)(inverse ? acc / ((double)n * n) : acc);
        }
}

/* Textbook iterative radix-2 decimation-in-time FFT of n (power of two) points with stride,
 * in place, no scaling.  w[k] = exp(-+2 pi i k / n), k < n/2. */
static void fft1(int n, cplx *x, long stride, const cplx *w) {
    for (int i = 1, j = 0; i < n; ++i) { /* bit-reversal permutation */
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { cplx t = x[i * stride]; x[i * stride] = x[j * stride]; x[j * stride] = t; }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1, tw = n / len;
        for (int s = 0; s < n; s += len)
            for (int k = 0; k < half; ++k) {
                cplx a = x[(s + k) * stride], b = x[(s + k + half) * stride] * w[k * tw];
                x[(s + k) * stride] = a + b;
                x[(s + k + half) * stride] = a - b;
            }
    }
}

/* 2-D transform of an n x n row-major array in place: rows, then columns. */
void orc_fft2(int n, cplx *a, int inverse) {
    cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)(n / 2 + 1));
    for (int k = 0; k < n / 2; ++k) {
        double ang = (inverse ? 2.0 : -2.0) * M_PI * k / n;
        w[k] = (cplx)(cos(ang) + I * sin(ang));
    }
    for (int y = 0; y < n; ++y) fft1(n, a + (size_t)y * n, 1, w);
    for (int x = 0; x < n; ++x) fft1(n, a + x, n, w);
    if (inverse) {
        const real s = (real)1 / ((real)n * (real)n);
        for (long i = 0; i < (long)n * n; ++i) a[i] *= s;
    }
    free(w);
}

/* ------------------------------------------------------------------------------------------
 * C2 modulus projection of the K modes of one frame (readings R2, R3, R6).
 * Phi, out: K x n x n.  Inten: n x n, negative = masked ("no constraint").  Returns the frame's
 * error term  sum_q (sqrt(I) - A)^2  over unmasked pixels, A = sqrt(sum_k |Phi_k|^2)  (C3).
 * pbound > 0: relaxed form; e = that sum / n^2; e <= pbound -> identity; else r = sqrt(pbound/e)
 * and Phi'_k = Phi_k * ((1 - r) sqrt(I)/A + r).  A == 0 (R2): mode 0 gets the modulus with zero
 * phase, the others 0 (then blended with r like every other pixel).
 * ------------------------------------------------------------------------------------------ */
real orc_modulus_project(int n, int K, const cplx *Phi, const real *Inten, real pbound, cplx *out) {
    const long np = (long)n * n;
    real *A = (real *)malloc(sizeof(real) * (size_t)np);
    real err = 0;
    for (long q = 0; q < np; ++q) {
        real s = 0;
        for (int k = 0; k < K; ++k) s += CABS2(Phi[k * np + q]);
        A[q] = SQRT(s);
        if (Inten[q] >= 0) { real d = SQRT(Inten[q]) - A[q]; err += d * d; }
    }
    real r = 0;
    if (pbound > 0) {
        real e = err / (real)np;
        r = (e <= pbound) ? (real)1 : SQRT(pbound / e);
    }
    for (long q = 0; q < np; ++q)
        for (int k = 0; k < K; ++k) {
            cplx z = Phi[k * np + q];
            if (Inten[q] < 0 || r == (real)1) { out[k * np + q] = z; continue; }
            cplx exact;
            if (A[q] > 0) exact = z * (SQRT(Inten[q]) / A[q]);
            else exact = (k == 0) ? (cplx)SQRT(Inten[q]) : (cplx)0;
            out[k * np + q] = (pbound > 0) ? (((real)1 - r) * exact + r * z) : exact;
        }
    free(A);
    return err;
}

/* sum of I over unmasked pixels (denominator of C3) */
double orc_sum_intensity(long count, const real *Inten) {
    double s = 0;
    for (long i = 0; i < count; ++i) if (Inten[i] >= 0) s += Inten[i];
    return s;
}

/* C1 exit wave of frame j, all modes: psi_k = P_k * O[r_j + .]  (north_star "psi_j = P * O[r_j]") */
static void exit_wave(int W, int n, int K, const cplx *O, const cplx *P, const int32_t *pos_j, cplx *psi) {
    const long np = (long)n * n;
    for (int k = 0; k < K; ++k)
        for (int y = 0; y < n; ++y)
            for (int x = 0; x < n; ++x)
                psi[k * np + y * n + x] = P[k * np + y * n + x] * O[(long)(pos_j[0] + y) * W + pos_j[1] + x];
}

/* R7 eval_error: sum_j sum_q (sqrt I_j - A_j)^2 with A_j the amplitude of F[P O_j]. */
double orc_eval_error_num(int H, int W, int n, int K, int J, const cplx *O, const cplx *P,
                          const int32_t *pos, const real *Inten) {
    (void)H;
    const long np = (long)n * n;
    double *ej = (double *)calloc((size_t)J, sizeof(double));
#pragma omp parallel
    {
        cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)(K * np));
#pragma omp for schedule(dynamic, 4)
        for (int j = 0; j < J; ++j) {
            exit_wave(W, n, K, O, P, pos + 2 * j, w);
            for (int k = 0; k < K; ++k) orc_fft2(n, w + k * np, 0);
            double e = 0;
            for (long q = 0; q < np; ++q) {
                if (Inten[j * np + q] < 0) continue;
                real s = 0;
                for (int k = 0; k < K; ++k) s += CABS2(w[k * np + q]);
                real d = SQRT(Inten[j * np + q]) - SQRT(s);
                e += d * d;
            }
            ej[j] = e;
        }
        free(w);
    }
    double tot = 0;
    for (int j = 0; j < J; ++j) tot += ej[j];
    free(ej);
    return tot;
}

/* ------------------------------------------------------------------------------------------
 * DM, one iteration (SURVEY 8(c) "DM" steps 1-5, readings R4 (beta = 1, lagged probe sums),
 * R5 (blend regularisation), R6 (relaxed projection); north_star: "DM additionally applies the
 * reflector"; "keep a copy of the previous calculation in memory and calculate the
 * exit wavefronts of all the scan points at once").
 * State: O (H x W), P (K x n x n), psi (J x K x n x n), all updated in place.
 * eps_O, eps_P: the blend constants fixed at init (delta max|P0|^2, delta J max|O0|^2).
 * Returns sum_j sum_q (sqrt I - A)^2 with A the amplitude of the transformed (reflected) wave.
 * revised (optional, J x K x n x n): psi_F = F^-1[Pi_M F phi] of every frame.
 * ------------------------------------------------------------------------------------------ */
double orc_dm_iteration(int H, int W, int n, int K, int J, cplx *O, cplx *P, cplx *psi,
                        const int32_t *pos, const real *Inten, real eps_O, real eps_P,
                        int update_probe, real pbound, cplx *revised) {
    const long np = (long)n * n, knp = K * np;
    cplx *nP = (cplx *)calloc((size_t)knp, sizeof(cplx));
    real *dP = (real *)calloc((size_t)np, sizeof(real));
    cplx *nO = (cplx *)calloc((size_t)H * W, sizeof(cplx));
    real *dO = (real *)calloc((size_t)H * W, sizeof(real));
    double *ej = (double *)calloc((size_t)J, sizeof(double));

    /* step 1: lagged probe sums from the INCOMING psi_j and the current O */
    for (int j = 0; j < J; ++j) {
        const int32_t *r = pos + 2 * j;
        for (int y = 0; y < n; ++y)
            for (int x = 0; x < n; ++x) {
                cplx Oj = O[(long)(r[0] + y) * W + r[1] + x];
                for (int k = 0; k < K; ++k)
                    nP[k * np + y * n + x] += conj(Oj) * psi[j * knp + k * np + y * n + x];
                dP[y * n + x] += CABS2(Oj);
            }
    }

    /* steps 2-3 for every frame (independent given O, P) */
#pragma omp parallel
    {
        cplx *psiO = (cplx *)malloc(sizeof(cplx) * (size_t)knp);
        cplx *phi = (cplx *)malloc(sizeof(cplx) * (size_t)knp);
        cplx *prj = (cplx *)malloc(sizeof(cplx) * (size_t)knp);
#pragma omp for schedule(dynamic, 4)
        for (int j = 0; j < J; ++j) {
            cplx *pj = psi + j * knp;
            exit_wave(W, n, K, O, P, pos + 2 * j, psiO);               /* psi_O = P O_j          */
            for (long i = 0; i < knp; ++i) phi[i] = (real)2 * psiO[i] - pj[i];   /* reflector    */
            for (int k = 0; k < K; ++k) orc_fft2(n, phi + k * np, 0);  /* Phi = F[phi]           */
            ej[j] = orc_modulus_project(n, K, phi, Inten + j * np, pbound, prj); /* Phi' = Pi_M  */
            for (int k = 0; k < K; ++k) orc_fft2(n, prj + k * np, 1);  /* psi_F = F^-1[Phi']     */
            if (revised) memcpy(revised + j * knp, prj, sizeof(cplx) * (size_t)knp);
            for (long i = 0; i < knp; ++i) pj[i] = pj[i] + prj[i] - psiO[i];   /* step 3, beta=1 */
        }
        free(psiO); free(phi); free(prj);
    }

    /* step 4: object sums from the NEW psi_j */
    for (int j = 0; j < J; ++j) {
        const int32_t *r = pos + 2 * j;
        for (int y = 0; y < n; ++y)
            for (int x = 0; x < n; ++x) {
                long o = (long)(r[0] + y) * W + r[1] + x;
                for (int k = 0; k < K; ++k) {
                    cplx Pk = P[k * np + y * n + x];
                    nO[o] += conj(Pk) * psi[j * knp + k * np + y * n + x];
                    dO[o] += CABS2(Pk);
                }
            }
    }

    /* step 5: blended divisions (R5) */
    for (long o = 0; o < (long)H * W; ++o) O[o] = (nO[o] + eps_O * O[o]) / (dO[o] + eps_O);
    if (update_probe)
        for (int k = 0; k < K; ++k)
            for (long q = 0; q < np; ++q)
                P[k * np + q] = (nP[k * np + q] + eps_P * P[k * np + q]) / (dP[q] + eps_P);

    double tot = 0;
    for (int j = 0; j < J; ++j) tot += ej[j];
    free(nP); free(dP); free(nO); free(dO); free(ej);
    return tot;
}

/* ------------------------------------------------------------------------------------------
 * ePIE-minibatch and LSQML-style minibatch, one batch (SURVEY 8(c) "ePIE-minibatch",
 * "LSQML-style minibatch", readings R8, R9).  O and P are frozen while the batch's sums are
 * formed, then both are stepped from the pre-batch state.
 *   frames[0..nb): the frames of the batch, visited in this order.
 *   ePIE (alg 0): O += alpha_O dO, P_k += alpha_P dP_k.
 *   LSQML (alg 2): joint real step (a, b) minimising the linearised residual
 *       sum_{j,k} || chi_jk - a P_k dO_j - b dP_k O_j ||^2  with Tikhonov lambda on the diagonal,
 *     its five sums taken here from their per-frame DEFINITIONS (chi is kept for the batch).
 *   dO = n_O / (d_O + delta_O max_r sum_k |P_k|^2),  dP_k = n_Pk / (d_P + delta_P max_r d_P).
 * step_out[0..1] = the (a, b) applied.  revised (optional): F^-1[Phi'] for the batch's frames,
 * indexed by position in `frames`.  Returns the batch's error term sum (sqrt I - A)^2.
 * ------------------------------------------------------------------------------------------ */
double orc_minibatch_step(int alg, int H, int W, int n, int K, cplx *O, cplx *P,
                          const int32_t *pos, const real *Inten, const int32_t *frames, int nb,
                          int update_probe, real alpha_O, real alpha_P, real delta_O, real delta_P,
                          real lsq_lambda, real pbound, double *step_out, cplx *revised) {
    const long np = (long)n * n, knp = K * np, HW = (long)H * W;
    cplx *chi = (cplx *)malloc(sizeof(cplx) * (size_t)(nb * knp));
    double *ej = (double *)calloc((size_t)nb, sizeof(double));
    cplx *nO = (cplx *)calloc((size_t)HW, sizeof(cplx));
    real *dO = (real *)calloc((size_t)HW, sizeof(real));
    cplx *nP = (cplx *)calloc((size_t)knp, sizeof(cplx));
    real *dP = (real *)calloc((size_t)np, sizeof(real));

#pragma omp parallel
    {
        cplx *psi = (cplx *)malloc(sizeof(cplx) * (size_t)knp);
        cplx *Phi = (cplx *)malloc(sizeof(cplx) * (size_t)knp);
#pragma omp for schedule(dynamic, 4)
        for (int i = 0; i < nb; ++i) {
            int j = frames[i];
            exit_wave(W, n, K, O, P, pos + 2 * j, psi);                 /* psi = P O_j           */
            memcpy(Phi, psi, sizeof(cplx) * (size_t)knp);
            for (int k = 0; k < K; ++k) orc_fft2(n, Phi + k * np, 0);   /* Phi = F[psi]          */
            cplx *c = chi + i * knp;
            ej[i] = orc_modulus_project(n, K, Phi, Inten + j * np, pbound, c);
            for (int k = 0; k < K; ++k) orc_fft2(n, c + k * np, 1);     /* F^-1[Pi_M Phi]        */
            if (revised) memcpy(revised + i * knp, c, sizeof(cplx) * (size_t)knp);
            for (long q = 0; q < knp; ++q) c[q] -= psi[q];              /* chi = ... - psi       */
        }
        free(psi); free(Phi);
    }

    /* batch sums, serial, in batch order (old O_j in the probe sums) */
    for (int i = 0; i < nb; ++i) {
        const int32_t *r = pos + 2 * frames[i];
        for (int y = 0; y < n; ++y)
            for (int x = 0; x < n; ++x) {
                long o = (long)(r[0] + y) * W + r[1] + x, q = y * n + x;
                cplx Oj = O[o];
                for (int k = 0; k < K; ++k) {
                    cplx Pk = P[k * np + q], c = chi[i * knp + k * np + q];
                    nO[o] += conj(Pk) * c;
                    dO[o] += CABS2(Pk);
                    nP[k * np + q] += conj(Oj) * c;
                }
                dP[q] += CABS2(Oj);
            }
    }

    /* preconditioned directions */
    real maxP = 0, maxdP = 0;
    for (long q = 0; q < np; ++q) {
        real s = 0;
        for (int k = 0; k < K; ++k) s += CABS2(P[k * np + q]);
        if (s > maxP) maxP = s;
        if (dP[q] > maxdP) maxdP = dP[q];
    }
    for (long o = 0; o < HW; ++o) nO[o] = nO[o] / (dO[o] + delta_O * maxP);        /* now Delta O   */
    for (int k = 0; k < K; ++k)
        for (long q = 0; q < np; ++q) nP[k * np + q] = nP[k * np + q] / (dP[q] + delta_P * maxdP); /* Delta P_k */

    double a = alpha_O, b = update_probe ? alpha_P : 0;
    if (alg == ALG_LSQML) {
        double A11 = 0, A22 = 0, A12 = 0, b1 = 0, b2 = 0;
        for (int i = 0; i < nb; ++i) {
            const int32_t *r = pos + 2 * frames[i];
            for (int k = 0; k < K; ++k)
                for (int y = 0; y < n; ++y)
                    for (int x = 0; x < n; ++x) {
                        long o = (long)(r[0] + y) * W + r[1] + x, q = k * np + y * n + x;
                        double complex u = (double complex)(P[q] * nO[o]);    /* P_k dO_j      */
                        double complex v = (double complex)(nP[q] * O[o]);    /* dP_k O_j      */
                        double complex c = (double complex)chi[i * knp + q];
                        A11 += creal(conj(u) * u); A22 += creal(conj(v) * v);
                        A12 += creal(conj(u) * v);
                        b1 += creal(conj(u) * c);  b2 += creal(conj(v) * c);
                    }
        }
        double l = 1.0 + (double)lsq_lambda;
        if (!update_probe) {
            a = (A11 > 0) ? b1 / (A11 * l) : 0; b = 0;
        } else {
            double det = A11 * l * A22 * l - A12 * A12;
            if (!(det > 0) || !isfinite(det)) { a = 0; b = 0; }
            else { a = (b1 * A22 * l - A12 * b2) / det; b = (A11 * l * b2 - A12 * b1) / det; }
        }
    }
    for (long o = 0; o < HW; ++o) O[o] += (real)a * nO[o];
    if (update_probe) for (long q = 0; q < knp; ++q) P[q] += (real)b * nP[q];
    if (step_out) { step_out[0] = a; step_out[1] = b; }

    double tot = 0;
    for (int i = 0; i < nb; ++i) tot += ej[i];
    free(chi); free(ej); free(nO); free(dO); free(nP); free(dP);
    return tot;
}

/* ------------------------------------------------------------------------------------------
 * Textbook (sequential) DM overlap projection, SURVEY 8(f) f1 / reading R4's alternative: after the
 * Fourier step the object is formed from the new psi_j with the current probe, THEN the probe from the
 * same psi_j with the NEW object, optionally repeated ("n inner sweeps").  PAPER.md:58 ("DM has to keep
 * a copy of the previous calculation ... calculate the exit wavefronts of all the scan points at once")
 * describes exactly this two-set alternation.  Both divisions are blended as in R5.
 *   orc_object_from_waves : O <- (sum_j sum_k conj(P_k) psi_jk + eps_O O) / (sum_j sum_k |P_k|^2 + eps_O)
 *   orc_probe_from_waves  : P_k <- (sum_j conj(O_j) psi_jk + eps_P P_k) / (sum_j |O_j|^2 + eps_P)
 * ------------------------------------------------------------------------------------------ */
void orc_object_from_waves(int H, int W, int n, int K, int J, cplx *O, const cplx *P, const cplx *psi,
                           const int32_t *pos, real eps_O) {
    const long np = (long)n * n, knp = K * np;
    cplx *nO = (cplx *)calloc((size_t)H * W, sizeof(cplx));
    real *dO = (real *)calloc((size_t)H * W, sizeof(real));
    for (int j = 0; j < J; ++j) {
        const int32_t *r = pos + 2 * j;
        for (int y = 0; y < n; ++y)
            for (int x = 0; x < n; ++x) {
                long o = (long)(r[0] + y) * W + r[1] + x;
                for (int k = 0; k < K; ++k) {
                    cplx Pk = P[k * np + y * n + x];
                    nO[o] += conj(Pk) * psi[j * knp + k * np + y * n + x];
                    dO[o] += CABS2(Pk);
                }
            }
    }
    for (long o = 0; o < (long)H * W; ++o) O[o] = (nO[o] + eps_O * O[o]) / (dO[o] + eps_O);
    free(nO); free(dO);
}

void orc_probe_from_waves(int H, int W, int n, int K, int J, const cplx *O, cplx *P, const cplx *psi,
                          const int32_t *pos, real eps_P) {
    (void)H;
    const long np = (long)n * n, knp = K * np;
    cplx *nP = (cplx *)calloc((size_t)knp, sizeof(cplx));
    real *dP = (real *)calloc((size_t)np, sizeof(real));
    for (int j = 0; j < J; ++j) {
        const int32_t *r = pos + 2 * j;
        for (int y = 0; y < n; ++y)
            for (int x = 0; x < n; ++x) {
                cplx Oj = O[(long)(r[0] + y) * W + r[1] + x];
                for (int k = 0; k < K; ++k)
                    nP[k * np + y * n + x] += conj(Oj) * psi[j * knp + k * np + y * n + x];
                dP[y * n + x] += CABS2(Oj);
            }
    }
    for (int k = 0; k < K; ++k)
        for (long q = 0; q < np; ++q)
            P[k * np + q] = (nP[k * np + q] + eps_P * P[k * np + q]) / (dP[q] + eps_P);
    free(nP); free(dP);
}

/* ------------------------------------------------------------------------------------------
 * LSQML-style minibatch with PER-FRAME step lengths (reading R25; ref [18] of the paper
 * is not available, so this is a definition in the spirit of R9, not a reproduction).  Directions dO, dP_k
 * as in orc_minibatch_step.  For every frame j of the batch the real pair (a_j, b_j) minimises
 *     sum_k || chi_jk - a_j P_k dO_j - b_j dP_k O_j ||^2  + lambda (A11_j a_j^2 + A22_j b_j^2)
 * (2x2 normal equations; frozen probe: a_j = b1_j / (A11_j (1 + lambda)), b_j = 0; determinant <= 0: 0, 0).
 * Update ("weighted second scatter"): with w_j(r) = sum_k |P_k(r - r_j)|^2 on the frame's window,
 *     O(r) += dO(r) * sum_j a_j w_j(r) / sum_j w_j(r)     (pixels with sum_j w_j = 0 keep their value)
 *     P_k  += mean_j(b_j) * dP_k.
 * steps_out (optional): nb pairs (a_j, b_j), in batch order.  Returns the batch's error term.
 * ------------------------------------------------------------------------------------------ */
double orc_minibatch_step_perframe(int H, int W, int n, int K, cplx *O, cplx *P, const int32_t *pos, const real *Inten,
                                   const int32_t *frames, int nb, int update_probe, real delta_O, real delta_P,
                                   real lsq_lambda, real pbound, double *steps_out) {
    const long np = (long)n * n, knp = K * np, HW = (long)H * W;
    cplx *chi = (cplx *)malloc(sizeof(cplx) * (size_t)(nb * knp));
    cplx *psi = (cplx *)malloc(sizeof(cplx) * (size_t)knp);
    cplx *Phi = (cplx *)malloc(sizeof(cplx) * (size_t)knp);
    cplx *nO = (cplx *)calloc((size_t)HW, sizeof(cplx));
    real *dO = (real *)calloc((size_t)HW, sizeof(real));
    cplx *nP = (cplx *)calloc((size_t)knp, sizeof(cplx));
    real *dP = (real *)calloc((size_t)np, sizeof(real));
    double tot = 0;
    for (int i = 0; i < nb; ++i) {                                      /* chi_j = F^-1[Pi_M F[P O_j]] - P O_j */
        int j = frames[i];
        exit_wave(W, n, K, O, P, pos + 2 * j, psi);
        memcpy(Phi, psi, sizeof(cplx) * (size_t)knp);
        for (int k = 0; k < K; ++k) orc_fft2(n, Phi + k * np, 0);
        cplx *c = chi + i * knp;
        tot += orc_modulus_project(n, K, Phi, Inten + j * np, pbound, c);
        for (int k = 0; k < K; ++k) orc_fft2(n, c + k * np, 1);
        for (long q = 0; q < knp; ++q) c[q] -= psi[q];
    }
    for (int i = 0; i < nb; ++i) {                                      /* batch sums (as in orc_minibatch_step) */
        const int32_t *r = pos + 2 * frames[i];
        for (int y = 0; y < n; ++y)
            for (int x = 0; x < n; ++x) {
                long o = (long)(r[0] + y) * W + r[1] + x, q = y * n + x;
                cplx Oj = O[o];
                for (int k = 0; k < K; ++k) {
                    cplx Pk = P[k * np + q], c = chi[i * knp + k * np + q];
                    nO[o] += conj(Pk) * c; dO[o] += CABS2(Pk); nP[k * np + q] += conj(Oj) * c;
                }
                dP[q] += CABS2(Oj);
            }
    }
    real maxP = 0, maxdP = 0;
    for (long q = 0; q < np; ++q) {
        real s = 0;
        for (int k = 0; k < K; ++k) s += CABS2(P[k * np + q]);
        if (s > maxP) maxP = s;
        if (dP[q] > maxdP) maxdP = dP[q];
    }
    for (long o = 0; o < HW; ++o) nO[o] = nO[o] / (dO[o] + delta_O * maxP);            /* dO direction */
    for (int k = 0; k < K; ++k)
        for (long q = 0; q < np; ++q) nP[k * np + q] = nP[k * np + q] / (dP[q] + delta_P * maxdP);

    double *aw = (double *)calloc((size_t)HW, sizeof(double)), *ww = (double *)calloc((size_t)HW, sizeof(double));
    double bsum = 0;
    const double l = 1.0 + (double)lsq_lambda;
    for (int i = 0; i < nb; ++i) {                                      /* per-frame 2x2 solves */
        const int32_t *r = pos + 2 * frames[i];
        double A11 = 0, A22 = 0, A12 = 0, b1 = 0, b2 = 0;
        for (int k = 0; k < K; ++k)
            for (int y = 0; y < n; ++y)
                for (int x = 0; x < n; ++x) {
                    long o = (long)(r[0] + y) * W + r[1] + x, q = k * np + y * n + x;
                    double complex u = (double complex)(P[q] * nO[o]), v = (double complex)(nP[q] * O[o]);
                    double complex c = (double complex)chi[i * knp + q];
                    A11 += creal(conj(u) * u); A22 += creal(conj(v) * v); A12 += creal(conj(u) * v);
                    b1 += creal(conj(u) * c); b2 += creal(conj(v) * c);
                }
        double a, b;
        if (!update_probe) { a = (A11 > 0) ? b1 / (A11 * l) : 0; b = 0; }
        else {
            double det = A11 * l * A22 * l - A12 * A12;
            if (!(det > 0) || !isfinite(det)) { a = 0; b = 0; }
            else { a = (b1 * A22 * l - A12 * b2) / det; b = (A11 * l * b2 - A12 * b1) / det; }
        }
        if (steps_out) { steps_out[2 * i] = a; steps_out[2 * i + 1] = b; }
        bsum += b;
        for (int y = 0; y < n; ++y)                                      /* weighted second scatter */
            for (int x = 0; x < n; ++x) {
                long o = (long)(r[0] + y) * W + r[1] + x;
                double w = 0;
                for (int k = 0; k < K; ++k) w += (double)CABS2(P[k * np + y * n + x]);
                aw[o] += a * w; ww[o] += w;
            }
    }
    for (long o = 0; o < HW; ++o) if (ww[o] > 0) O[o] += (real)(aw[o] / ww[o]) * nO[o];
    if (update_probe) { real bm = (real)(bsum / nb); for (long q = 0; q < knp; ++q) P[q] += bm * nP[q]; }
    free(chi); free(psi); free(Phi); free(nO); free(dO); free(nP); free(dP); free(aw); free(ww);
    return tot;
}
