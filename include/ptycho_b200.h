/* ptycho_b200.h -- C ABI of the B200-native ptychographic projection cycle.
 *
 * The calls follow the paper's step-mode API  init / step / fetch object / fetch probe / post
 * (PAPER.md:96 and Listing 1: epieinit, epiestep, epieresobj, epieresprobe,
 * epiepost; "analogous calls for DM and LSQML", Fig. 3) and BASELINE.json north_star:
 * "init(object, probe, positions, intensities), iterate(algorithm, n), fetch object/probe/error".
 * The state (object, probe, exit waves) stays on the GPU between calls and can be fetched at
 * any iteration.  The shape of this header is SURVEY.md section 8(b).
 *
 * Notation: N frame side, J scan positions, K probe modes, object O
 * (H x W), probe P_k (N x N), position r_j = (y_j, x_j) = top-left corner of the patch,
 * O_j = O[y_j : y_j+N, x_j : x_j+N], I_j measured intensity (N x N, >= 0, FFT order: DC at
 * [0,0]).  F = unnormalised forward 2-D DFT, F^-1 carries 1/N^2 (reading R1).  All complex
 * arrays are interleaved complex64 (re, im), row-major.
 *
 * Pointers: every data pointer may be HOST or DEVICE memory (detected with
 * cudaPointerGetAttributes) unless stated.  `workspace` must be DEVICE memory.
 * Threading: one context is used from one host thread at a time.
 * Errors: every call returns a status; nothing is thrown across the ABI; a call that returns
 * an error leaves the context unchanged (except PTYCHO_ECUDA, after which the context should
 * be destroyed).  ptycho_last_error() gives a message for the last failing call.
 */
#ifndef PTYCHO_B200_H
#define PTYCHO_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ptycho_ctx ptycho_ctx; /* opaque; owned by the library */

typedef enum {
    PTYCHO_OK = 0,
    PTYCHO_EINVAL = 1,       /* null pointer, N not in {64,128,256,512}, K < 1, J < 1, bad parameter */
    PTYCHO_EBOUNDS = 2,      /* a position with y<0, x<0, y+N>H or x+N>W (no wrap, no clamp; R10)     */
    PTYCHO_EUNSUPPORTED = 3, /* K > PTYCHO_MAX_MODES                                                  */
    PTYCHO_ENOMEM = 4,       /* workspace smaller than ptycho_workspace_bytes()                       */
    PTYCHO_ECUDA = 5,        /* a CUDA runtime error; message in ptycho_last_error()                  */
    PTYCHO_ESTATE = 6        /* call not valid in the current state (e.g. exit waves before any DM)   */
} ptycho_status;

/* The three algorithms the paper's back end offers, in their data-parallel
 * forms: */
typedef enum {
    PTYCHO_EPIE_MB = 0, /* ePIE, minibatch form (reading R8)                             */
    PTYCHO_DM = 1,      /* difference map, all positions at once (reading R4) */
    PTYCHO_LSQML = 2,   /* LSQML-style minibatch with one joint step per batch (R9)       */
    PTYCHO_LSQML_PF = 3 /* the same directions, but one step pair (a_j, b_j) per FRAME and the weighted second scatter
                           O += dO sum_j a_j w_j / sum_j w_j, w_j = sum_k |P_k|^2 on the frame's window; P_k += mean_j(b_j) dP_k
                           (reading R25).  Costs a second transform cycle per batch (chi is recomputed,
                           not kept).  ptycho_fetch_steps then returns one pair per frame, batch after batch; inside a batch
                           in the library's own (spatially sorted) frame order                                       */
} ptycho_alg;

typedef enum {
    PTYCHO_I_F32 = 0, /* float32 counts; a negative value marks a masked pixel (R3)   */
    PTYCHO_I_U16 = 1  /* uint16 counts; 65535 marks a masked / saturated pixel (R3, R11) */
} ptycho_itype;

#define PTYCHO_MAX_MODES 8

/* Parameters; fill with ptycho_default_params() then override. */
typedef struct {
    int batch_size;     /* EPIE_MB / LSQML: frames per minibatch; 0 = all J (full batch)           */
    int probe_start;    /* first iteration (0-based, global counter) that updates the probe
                           ("after which iteration to update the probe")              */
    float delta_blend;  /* DM: blend regulariser delta of (n + eps x_old)/(d + eps)  (R5), 1e-2    */
    float delta_obj;    /* minibatch: dO = n_O/(d_O + delta_obj  * max_r sum_k|P_k|^2) (R8), 1.0   */
    float delta_probe;  /* minibatch: dP = n_P/(d_P + delta_probe* max_r d_P)          (R8), 1.0   */
    float alpha_obj;    /* EPIE_MB step on dO, 1.0                                                 */
    float alpha_probe;  /* EPIE_MB step on dP, 1.0                                                 */
    float lsq_lambda;   /* LSQML Tikhonov factor on the 2x2 diagonal (R9), 0.1                     */
    float pbound;       /* relaxed modulus projection: per-frame power bound, mean squared
                           amplitude error per pixel in counts; 0 = exact projection (R6)          */
    int disable_dm;     /* 1 = do not reserve the DM exit-wave store (J*K*N*N complex64) in the
                           workspace; ptycho_iterate(PTYCHO_DM) then returns PTYCHO_ESTATE          */
    int deterministic;  /* 1 = fixed-order gather accumulation of the overlap sums (north_star "deterministic
                           sorted-tile mode"): O, P and psi are bit-reproducible run to run; psi is read
                           twice more per iteration.  Single-mode DM only: init returns
                           PTYCHO_EUNSUPPORTED for n_modes > 1 or disable_dm, iterate for the minibatch
                           algorithms.  0 = atomic scatter-add                                     */
    int dm_sweeps;      /* DM overlap projection.  0 = reading R4: probe sums taken from the incoming exit waves (lagged),
                           one pass over the exit waves per iteration.  n >= 1 = the textbook sequential form (SURVEY.md
                           8(f) f1): object from the new exit waves, then the probe from the same waves and
                           the NEW object, n sweeps; the exit waves are read once more per sweep (twice from the second
                           sweep on).  Single-mode DM only (PTYCHO_EUNSUPPORTED otherwise)                        */
    const int32_t *batch_order; /* HOST pointer or NULL.  NULL: strided batches, n_b = ceil(J/B),
                           batch b = { j : j mod n_b = b } (R8).  Else a permutation of 0..J-1;
                           batch b = its entries [b*B, (b+1)*B).  Copied at init.                  */
    /* One scan over several GPUs.  shard_total_pos > 0 makes the context a SHARD:
       it holds n_pos of the scan's shard_total_pos frames and is driven by ptycho_shard_begin / ptycho_shard_end below.     */
    int shard_total_pos;        /* 0 = an ordinary context.  Else J of the WHOLE scan (eps_P = delta J max|O|^2, R5)          */
    int n_foreign;              /* number of entries of foreign_pos                                                          */
    const int32_t *foreign_pos; /* HOST pointer or NULL: (y, x) of the frames held by OTHER shards that overlap the object rows
                                   this shard's frames cover.  They enter d_O = sum_j |P(q - r_j)|^2 only (which needs the probe
                                   and the positions, not the frames' data).  Copied at init.                                */
    /* Sub-pixel scan positions (reading R28 -- PAPER.md does not say how the fractional part of a position
       is treated, so the textbook rule is taken: the Fourier shift theorem applied to the probe).                            */
    const float *subpixel_yx;   /* HOST pointer or NULL: n_pos x (dy, dx), each in [0, 1): frame j sits at pos_yx[j] + (dy, dx).  It sees
                                   the probe P_jk = S_d[P_k] = F^-1[F[P_k] exp(-2 pi i (k_y dy + k_x dx)/N)] (k signed, Nyquist = -N/2),
                                   the object patch stays at the integer corner; object sums use conj(P_jk), |P_jk|^2; the probe term
                                   conj(O_j) chi_jk is shifted back by S_{-d} before it is summed; d_P = sum_j |O_j|^2 and the object
                                   regulariser delta_obj max_r sum_k |P_k|^2 use unshifted quantities.  PTYCHO_EPIE_MB, PTYCHO_LSQML (the joint step's
                                   sums A22, A12 are then taken per frame with the shifted probe direction S_d[dP_k]) and PTYCHO_DM (through
                                   the three-pass kernels: the persistent DM kernel shares one probe among frames; the lagged probe
                                   terms conj(O_j) psi_jk are shifted back like the minibatch ones); ptycho_iterate
                                   returns PTYCHO_EUNSUPPORTED for PTYCHO_LSQML_PF, ptycho_revised_waves likewise (ptycho_eval_error works:
                                   the data-fit error with the shifted probes); init returns it with deterministic, dm_sweeps or shard_total_pos.  Two more 2-D FFTs per
                                   frame and mode, one launch-sized buffer of per-frame probes in the workspace.  Copied at init.  */
} ptycho_params;

void ptycho_default_params(ptycho_params *p);

/* Bytes of device workspace ptycho_init needs for these sizes (0 on invalid sizes).  It holds
 * O, P, the DM exit-wave store (J*K*N*N complex64), the overlap canvases, the transform scratch,
 * the sort tables and, if the intensities are passed from host memory AND disable_dm is set, a copy of them (otherwise the copy is staged in the exit-wave store during init)
 * (`intensities_on_host`: 0 = device pointer, 1 = host pointer, 2 = none at init: streaming context, see ptycho_append_frames). */
size_t ptycho_workspace_bytes(int obj_h, int obj_w, int n, int n_modes, int n_pos,
                              ptycho_itype itype, int intensities_on_host,
                              const ptycho_params *params /* NULL = defaults */);

/* Create a context.  object: obj_h*obj_w complex64; probe: n_modes*n*n complex64; pos_yx:
 * n_pos*(y,x) int32 top-left corners; intensities: n_pos*n*n of `itype` in FFT order.
 * object, probe and positions are COPIED.  intensities are BORROWED when the pointer is device
 * memory (it must outlive the context) and copied into the workspace when it is host memory.
 * workspace: device memory of at least ptycho_workspace_bytes(), 256-byte aligned, owned by the
 * caller, must outlive the context.  cuda_stream: a cudaStream_t (NULL = default stream); all
 * work of this context is issued on it.  Fixes the DM blend constants from the initial state:
 * eps_O = delta max_r sum_k|P_k|^2, eps_P = delta J max|O|^2 (R5).  Synchronises the stream. */
ptycho_status ptycho_init(ptycho_ctx **out, const float *object, int obj_h, int obj_w,
                          const float *probe, int n_modes, int n, const int32_t *pos_yx, int n_pos,
                          const void *intensities, ptycho_itype itype, const ptycho_params *params,
                          void *workspace, size_t workspace_bytes, void *cuda_stream);

/* Run n_iters iterations of `alg` (one iteration = one pass over all J positions, R20).
 * Asynchronous: kernels are queued on the context's stream and the call returns.  The iteration
 * counter is global across calls (probe_start and the error history continue).  DM keeps the
 * exit waves psi_j; if they are not valid (first DM call, or a minibatch algorithm ran since)
 * they are first set to psi_j = P O_j (R4).  Per frame the cycle is: exit wave psi_O = P O_j
 * (DM: reflector 2 psi_O - psi_j), forward FFT, error term and modulus projection onto sqrt(I_j)
 * (relaxed when pbound > 0), inverse FFT, exit-wave update, overlap scatter-add of object and
 * probe sums, then the normalising update. */
ptycho_status ptycho_iterate(ptycho_ctx *ctx, ptycho_alg alg, int n_iters);

/* Copy the current state out (synchronises the stream).  out: host or device. */
ptycho_status ptycho_fetch_object(ptycho_ctx *ctx, float *out /* obj_h*obj_w*2 */);
ptycho_status ptycho_fetch_probe(ptycho_ctx *ctx, float *out /* n_modes*n*n*2 */);
/* Error history E_t = sum_j sum_q (sqrt I_j - A_j)^2 / sum_j sum_q I_j over unmasked pixels, A_j
 * the amplitude of the wave transformed in iteration t (R7, C3).  out: HOST, up to cap values;
 * *n_written = number of iterations run so far (may exceed cap). */
ptycho_status ptycho_fetch_error(ptycho_ctx *ctx, double *out, int cap, int *n_written);
/* Exit waves of `count` frames idx[0..count) (caller's frame numbering; idx is a HOST pointer).
 * After DM: the stored psi_j.  Otherwise PTYCHO_ESTATE.  out: count*n_modes*n*n*2 floats. */
ptycho_status ptycho_fetch_exit_waves(ptycho_ctx *ctx, const int32_t *idx, int count, float *out);
/* Revised waves psi_F = F^-1[Pi_M F[P O_j]] of the CURRENT object and probe for frames idx
 * (one forward/projection/inverse pass, no state change); used for teacher-forced parity of the
 * minibatch algorithms. */
ptycho_status ptycho_revised_waves(ptycho_ctx *ctx, const int32_t *idx, int count, float *out);
/* LSQML: the (a, b) steps applied so far, in batch order; out: HOST, up to cap pairs. */
ptycho_status ptycho_fetch_steps(ptycho_ctx *ctx, double *out_ab, int cap, int *n_written);

/* Overwrite state (teacher forcing, checkpoint restore).  Source: host or device. */
ptycho_status ptycho_set_object(ptycho_ctx *ctx, const float *object);
ptycho_status ptycho_set_probe(ptycho_ctx *ctx, const float *probe);
ptycho_status ptycho_set_exit_waves(ptycho_ctx *ctx, const float *psi /* n_pos*n_modes*n*n*2 */);

/* Data-fit error of the current O, P: the E above evaluated for F[P O_j] (one FFT pass, no
 * state change; R7).  Synchronises. */
ptycho_status ptycho_eval_error(ptycho_ctx *ctx, double *out);

/* ---- streaming ingestion ----
 * PAPER.md:9 ("several TB's of data per second ... processed in real time") and PAPER.md:29 (3 kHz frames, 6 GB/s raw data): the
 * frames of a scan arrive while the reconstruction already runs.  A context created with intensities == NULL (and a workspace
 * sized with intensities_on_host = 2) knows every position but holds no frame.  ptycho_append_frames hands over the next `count`
 * frames, first_frame == ptycho_frames_present(ctx) (acquisition order, no gaps; PTYCHO_EINVAL otherwise).  The call returns at
 * once: the host->device copy (through a 64 MB staging piece of the workspace), the re-tiling and the intensity sum run on a
 * copy stream of the context, so they overlap a ptycho_iterate that is in flight on the context's stream; `intensities` (host,
 * pinned for a truly asynchronous copy, or device) must stay valid until ptycho_wait_frames returns.  ptycho_iterate waits
 * (on the device) for the frames appended before the call and works on frames [0, present): the minibatch algorithms form their
 * batches over those frames (R8 with J = present); PTYCHO_DM needs every frame and returns PTYCHO_ESTATE earlier,
 * as do ptycho_eval_error and a call with no frame present. */
ptycho_status ptycho_append_frames(ptycho_ctx *ctx, int first_frame, int count, const void *intensities);
ptycho_status ptycho_wait_frames(ptycho_ctx *ctx);     /* blocks until every appended frame is on the device */
int ptycho_frames_present(const ptycho_ctx *ctx);

/* Probe-mode orthogonalisation (reading R26; PAPER.md:49 several probe modes).  The K modes are replaced by
 * P' = U P, U = V^H the unitary that diagonalises their Gram matrix G_ij = sum_r P_i(r) conj(P_j(r)) = V diag(lambda) V^H, lambda
 * descending; each eigenvector's phase is fixed by making its largest-magnitude component real and positive.  sum_k |P_k(r)|^2
 * is unchanged at every pixel, so the model intensities are unchanged; stored DM exit waves are mixed alike.  The Gram matrix is
 * formed on the device in double; the K x K eigenproblem (K <= 8) is solved on the host (cyclic Jacobi): the call synchronises
 * the stream.  K = 1: no-op. */
ptycho_status ptycho_orthogonalize_modes(ptycho_ctx *ctx);

/* Per-kernel-class device timing (SURVEY.md 8(d) "Evidence to collect"; bench.py's roofline
 * object).  ptycho_profile(ctx, 1) resets the totals and makes every later launch of this context
 * be bracketed by two cudaEvents on the context's stream; ptycho_profile(ctx, 0) stops that.
 * ptycho_profile_fetch synchronises the stream and returns, for one class, the summed device
 * time of its launches (ms) and their number since the last reset. */
typedef enum {
    PTYCHO_K_ROWS_FWD = 0, /* a1-a3: exit wave, reflector, forward row FFTs                      */
    PTYCHO_K_COLS = 1,     /* a3-a6: column FFTs, error, modulus projection, inverse column FFTs */
    PTYCHO_K_ROWS_INV = 2, /* a6-a9: inverse row FFTs, exit-wave update, overlap scatter-add     */
    PTYCHO_K_UPDATE = 3,   /* a10/a11: normalising updates, step solve, error sum                */
    PTYCHO_K_OTHER = 4,    /* initial exit waves, frame copies of fetch/set                      */
    PTYCHO_K_MEGA = 5,     /* a1-a9 of a whole DM iteration in one persistent kernel (dm_mega.cuh) */
    PTYCHO_KCLASS_COUNT = 6
} ptycho_kclass;
ptycho_status ptycho_profile(ptycho_ctx *ctx, int enable);
ptycho_status ptycho_profile_fetch(ptycho_ctx *ctx, int kclass, double *total_ms, long long *n_launches);

/* ---- one scan over several GPUs: the exchange step ("the overlapping size where the data is
 * shared between multiple GPUs", "the job could also run on multiple GPUs") ----
 * Reading R27: the frames are partitioned over the GPUs; every GPU holds the exit waves and intensities of its own frames (all
 * the bulk bytes) and a full-size object array of which it only ever touches the rows its frames cover.  Per DM iteration the
 * overlap sums are taken over ALL frames before the divisions, so the result is the single-GPU result up to summation order
 * (the paper's "share-frequency" > 1, an approximation it does not define, is not built).  What crosses GPUs per iteration: the
 * object correction canvas c on the rows two shards both cover (neighbour exchange), the probe sums n_P, d_P (3 N^2 floats,
 * all-reduce), and once the intensity sum.  The library does no communication: between the two calls below the CALLER adds the
 * other shards' values into the buffers ptycho_shard_buffers names (the Python package does it with torch.distributed over NCCL:
 * paper_2202_03144_b200/sharded.py).
 *   ptycho_shard_begin: one DM iteration up to the exchange (a1-a9 of this shard's frames: the megakernel).  Afterwards
 *       c_canvas holds this shard's part of c(q) = sum_j keep_j conj(P(q - r_j)) v_j(q - r_j) and probe_sums its part of n_P, d_P.
 *   ptycho_shard_end: a10 with the summed buffers: O += c / (d_O + eps_O) with d_O over own AND foreign positions, the probe
 *       blend, the error term of this shard's frames divided by *sum_I (so the scan's E_t is the sum of the shards' values).
 * Only for contexts made with shard_total_pos > 0; those refuse ptycho_iterate.  Single-mode DM, atomic-scatter mode, all frames
 * given at init (PTYCHO_EUNSUPPORTED otherwise at init).  PTYCHO_ESTATE when the two calls do not alternate. */
typedef struct {
    float *c_canvas;    /* device, obj_h * obj_w complex64, row-major: rows [row0, row1) can be non-zero                      */
    float *probe_sums;  /* device, 3 * n * n floats: n_P (n*n complex64) followed by d_P (n*n floats)                       */
    double *sum_I;      /* device, one double: sum of this shard's unmasked intensities; to be replaced by the scan's total
                           once, before the first ptycho_shard_begin                                                       */
    double *err_hist;   /* device: E_t of the iterations run so far (this shard's share once sum_I is the total)            */
    int row0, row1;     /* object rows covered by this shard's frames                                                       */
} ptycho_shard_bufs;
ptycho_status ptycho_shard_buffers(ptycho_ctx *ctx, ptycho_shard_bufs *out);
ptycho_status ptycho_shard_begin(ptycho_ctx *ctx);
ptycho_status ptycho_shard_end(ptycho_ctx *ctx);

/* Number of kernel launches issued by this context so far (for bench.py's gpu_launches). */
long long ptycho_launch_count(const ptycho_ctx *ctx);

const char *ptycho_last_error(const ptycho_ctx *ctx); /* never NULL; "" if none; ctx == NULL: the last failing ptycho_init */
void ptycho_destroy(ptycho_ctx *ctx);                 /* frees host state; the workspace is the caller's */

/* ---- init-time preparation of raw detector frames (first item beyond the hot path) ----
 * PAPER.md:50 lists what the paper does to the diffraction patterns before reconstruction: their centre
 * is located, they are cropped to the reconstruction size, a noise threshold is applied and saturated
 * pixels are detected from the detector bit depth.  This call does that on the GPU and writes the
 * intensities in the layout ptycho_init takes (reading R1: FFT order, DC at [0,0]; reading R3: masked
 * pixels carry the sentinel 65535 (uint16) or -1 (fp32)).  For output pixel (ky, kx), 0 <= ky, kx < n:
 *     dy = ky < n/2 ? ky : ky - n,   dx = kx < n/2 ? kx : kx - n        (offset from the centre pixel)
 *     (uy, ux) = (dy, dx), (dx, -dy), (-dy, -dx), (-dx, dy) for rot90 = 0, 1, 2, 3: the pattern turned counter-clockwise by
 *                rot90 quarter turns about the centre pixel ("the rotation angles of the diffraction patterns";
 *                multiples of 90 degrees only, reading R23: any other angle needs an interpolation rule the paper does not give)
 *     sy = center_y + uy,   sx = center_x + ux
 *     v  = raw[frame][sy][sx]            (a source pixel outside the detector, or a raw value that already is
 *                                         the sentinel -- 65535 in uint16, negative in fp32: masked)
 *     saturation > 0 and v >= saturation : masked
 *     threshold  > 0 and v <  threshold  : 0
 *     otherwise v
 *     frame_scale != NULL: v <- v * frame_scale[frame] in fp32 ("diffraction pattern normalization"; reading R24:
 *                one factor per frame, e.g. monitor / exposure normalisation, applied after the threshold; masks are decided
 *                on the raw counts)
 *     uint16 output: rounded to nearest (ties to even), clipped to 65534
 * raw: n_frames x det_h x det_w, uint16 or fp32, row-major, host or device; out: n_frames x n x n, host or
 * device; n is any even size >= 2 (not only the FFT sizes).  Integer / byte work: results are bit-exact
 * against the oracle.  Synchronises the stream before returning.  PTYCHO_EINVAL on null pointers, odd n,
 * non-positive sizes, rot90 outside 0..3 or unknown types. */
ptycho_status ptycho_prepare_frames(const void *raw, ptycho_itype raw_type, int n_frames, int det_h, int det_w,
                                    int center_y, int center_x, int n, float threshold, float saturation,
                                    int rot90, const float *frame_scale /* n_frames floats, host or device, or NULL */,
                                    void *out, ptycho_itype out_type, void *cuda_stream);

/* Unit-test entry points of single kernels (tier T2).  Device pointers. */
/* Batched 2-D complex64 FFT of `count` n x n frames, in place, on `cuda_stream`. */
ptycho_status ptycho_test_fft2(float *data, int n, int count, int inverse, void *cuda_stream);

/* ---- an entry point that allocates nothing ----
 * Some callers cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it.
 * ptycho_test_fft2 above gets the scratch of its kernels (the forward and inverse twiddle tables of the line FFT, fft_core.cuh)
 * from cudaMalloc and fills it from the host.  This variant keeps that scratch in a file-scope device array of the library,
 * 2 * PTYCHO_NOALLOC_MAX_N complex64 = 8 KB, which every GPU that loads the library holds until the process exits; the tables are
 * written on the device (fp64 sine / cosine rounded to fp32, like the host's), so the call does no host-to-device copy either.
 * The same batched in-place 2-D complex64 FFT of `count` n x n frames (n = 64, 128, 256 or 512; the inverse is scaled by 1/n^2;
 * DC at [0][0]), same kernels, results within the FFT tolerance of ptycho_test_fft2 (2e-6 relative L2; bit-identical whenever the
 * device's and the host's fp64 sine agree after rounding to fp32).
 *   data: DEVICE pointer, count * n * n complex64, read and written.  cuda_stream: a cudaStream_t of the CURRENT device.
 *   ASYNCHRONOUS: the work is queued on the stream and the call returns; it calls no cudaMalloc, cudaFree, or allocating library
 *   routine, and does not synchronise.
 *   n > PTYCHO_NOALLOC_MAX_N: PTYCHO_ENOMEM ("exceeds the static scratch"); other invalid arguments: PTYCHO_EINVAL; the message
 *   is at ptycho_last_error(NULL).
 *   The scratch is SHARED by all calls on a device and keeps the last call's tables: every call rewrites the part it uses, in
 *   stream order, before its kernels read it.  Calls that overlap on the GPU (different streams, or several host threads on
 *   different streams) with DIFFERENT n race on it; serialise them (one stream, or events). */
#define PTYCHO_NOALLOC_MAX_N 512
ptycho_status ptycho_fft2_noalloc(float *data, int n, int count, int inverse, void *cuda_stream);

/* ---- micro-benchmark entry point: DFT-as-GEMM against the packed-fp32 line FFT (BASELINE.json north_star) ----
 * The forward 1-D FFT of every ROW of `count` n x n complex64 frames, in place, unscaled, natural order.
 *   impl 0: the row pass of the product kernels (register-blocked packed-fp32 line FFT, one shared-memory exchange); n = 64..512.
 *   impl 1: the same transform as two radix-16 stages on the tensor cores, one warp per line, no shared memory
 *           (csrc/fft_mma.cuh: mma.sync m16n8k8 TF32 with a 3-term split, fp32 accumulation); n = 256 only.
 * data: DEVICE pointer.  Asynchronous on cuda_stream (time it with events); allocates nothing (uses the static scratch of
 * ptycho_fft2_noalloc for the twiddles of impl 0: the same sharing rules apply).  PTYCHO_EUNSUPPORTED for other n, PTYCHO_EINVAL
 * for bad arguments.  Not used by any product path. */
ptycho_status ptycho_test_fft_rows(float *data, int n, int count, int impl, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* PTYCHO_B200_H */
