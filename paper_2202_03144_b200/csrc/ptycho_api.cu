// ptycho_api.cu -- host side of the C ABI declared in include/ptycho_b200.h.
//
// Holds no arithmetic of the method except the sequencing of iterations, chunks and minibatches
// (readings R4, R8, R20); every step of the cycle runs in the kernels of
// kernels.cuh.  There is no CPU fallback: without a CUDA device every call fails with
// PTYCHO_ECUDA.
#include "../../include/ptycho_b200.h"

#include <algorithm>
#include <cmath>
#include <complex>
#include <mutex>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <numeric>
#include <string>
#include <vector>

#include "kernels.cuh"
#include "dm_mega.cuh"
#include "dm_det.cuh"
#include "fft_mma.cuh"

using namespace ptycho;

namespace {

constexpr int kErrCap = 1 << 16;    // iterations of error history kept
constexpr int kStepCap = 1 << 18;   // (a, b) pairs kept
constexpr int kCrossParts = 8;      // blocks per frame of the LSQML cross-term gather
constexpr int kRedBlocks = 4736;    // blocks of the canvas reductions / element-wise kernels

struct Carver {                     // bump allocator over the caller's workspace (256-byte aligned)
    char* base;
    size_t off = 0;
    explicit Carver(void* b) : base(static_cast<char*>(b)) {}
    template <class T> T* take(size_t count) {
        off = (off + 255) & ~size_t(255);
        T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
        off += count * sizeof(T);
        return p;
    }
};

}  // namespace

struct ptycho_ctx {
    int H = 0, W = 0, N = 0, K = 0, J = 0, itype = 0;
    ptycho_params par{};
    cudaStream_t stream = nullptr;
    // device state (inside the workspace)
    float2 *O = nullptr, *P = nullptr, *psi = nullptr, *S = nullptr, *nO = nullptr, *nP = nullptr;
    float *dO = nullptr, *dP = nullptr, *e_part = nullptr, *e_tmp = nullptr;
    float2 *tw = nullptr, *twi = nullptr;
    YX* pos = nullptr;
    int *tile_start = nullptr, *tile_mid = nullptr, *tile_list = nullptr;   // frames per object tile (CSR; see ptycho_init)
    int* tile_slots = nullptr;                 // dm_sweeps > 0: the same CSR with slots as entries, ascending (k_det_object)
    float4* det_partial = nullptr;
    int det_tx = 0, det_ty = 0;
    void* It = nullptr;                        // intensities re-tiled for the DM megakernel
    YX* spos = nullptr;                        // positions in DM slot order
    int *dm_frames = nullptr, *mb_frames = nullptr, *tmp_idx = nullptr, *slot_of = nullptr;
    Scalars* sc = nullptr;
    double *err_hist = nullptr, *steps = nullptr, *partO = nullptr, *partP = nullptr, *partX = nullptr, *scratch_d = nullptr;
    const void* I = nullptr;
    // host state
    int chunk = 1;
    // DM megakernel (dm_mega.cuh): frames per wave, wave lag between passes, ring slots, grid
    int mega_M = 0, mega_D = 0, mega_R = 0, mega_grid = 0;
    int* mega_ctr = nullptr;                   // device: [head | pad to 64 ints | cnt1[J] | cnt2[J] | cnt3[J]]
    float* p2 = nullptr;                       // |P|^2 of the current probe (d_O gather, dm_det.cuh)
    float* wO = nullptr;                       // LSQML_PF: sum_j w_j canvas (the a_j w_j canvas reuses dO)
    float2* lsqT = nullptr;                    // LSQML: sum_k conj(P_k) dP_k of the current batch (k_lsq_T)
    double* pf_part = nullptr; float2* pf_ab = nullptr;   // LSQML_PF: per-frame partial sums (J x NCB x 5) and steps (J)
    double* err_part = nullptr; unsigned int* err_ticket = nullptr;   // k_sum_error: per-CTA pieces and the finishing ticket
    int* dm_stat = nullptr;                    // [0] frames inside the power bound in the previous DM iteration, [1] running count
    int sms = 148;
    std::vector<int> dm_order;                 // slot -> caller frame
    std::vector<int> slot_of_h;                // caller frame -> slot
    std::vector<int> mb_offsets;               // batch b = mb_frames[mb_offsets[b] .. mb_offsets[b+1])
    int t = 0;                                 // global iteration counter
    // streaming ingestion (ptycho_append_frames): frames [0, present) have arrived; the copies run on their own stream
    bool streaming = false;
    int present = 0, mb_built_for = -1, stage_frames = 0;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_append = nullptr;
    void* stage = nullptr;                     // device staging piece of the H2D copies
    double* scratch_s = nullptr;               // partial sums of the appended chunk's intensities (copy stream)
    std::vector<int32_t> pos_h;                // positions, caller order (batch rebuilds)
    std::vector<int> batch_order_h, mb_h;
    long long n_steps = 0;
    bool psi_valid = false;
    int epie_pi = -1;                          // ePIE-minibatch: which sc->max_p2s slot holds the current probe's maximum (-1: none, k_probe_max runs)
    // sub-pixel positions (params.subpixel_yx, R28): fractions (device, caller numbering), F[P], Fourier-space probe numerator,
    // per-frame probes of one launch
    float* sub_frac = nullptr;
    float2 *sub_FP = nullptr, *sub_nPF = nullptr, *sub_Pj = nullptr;
    float2 *sub_FdP = nullptr, *sub_dPj = nullptr;   // LSQML: F[dP] and the per-frame shifted probe directions of one launch
    double* partA22 = nullptr;
    std::vector<float> sub_frac_h;
    // shard of a scan held by several GPUs (ptycho_shard_begin / _end): positions of the other shards' frames over our rows
    std::vector<int32_t> foreign_h;
    bool shard_open = false;                   // between ptycho_shard_begin and ptycho_shard_end
    int shard_row0 = 0, shard_row1 = 0;
    long long launches = 0;
    std::string err;
    // per-kernel-class CUDA-event timing (ptycho_profile): (class, start, stop) of every launch
    bool prof = false;
    struct ProfEv { int cls; cudaEvent_t a, b; };
    std::vector<ProfEv> prof_ev;
    double prof_ms[PTYCHO_KCLASS_COUNT] = {};
    long long prof_n[PTYCHO_KCLASS_COUNT] = {};
    ~ptycho_ctx() {
        for (auto& e : prof_ev) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
        if (ev_append) cudaEventDestroy(ev_append);
        if (copy_stream) cudaStreamDestroy(copy_stream);
    }
};

namespace {

#define CU(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) {                                                                   \
            if (c) c->err = std::string(#call) + ": " + cudaGetErrorString(e_);                    \
            return PTYCHO_ECUDA;                                                                   \
        }                                                                                          \
    } while (0)

std::string g_init_error;   // message of the last failing ptycho_init (no context exists to hold it): ptycho_last_error(NULL)

ptycho_status fail(ptycho_ctx* c, ptycho_status s, const char* msg) {
    if (c) c->err = msg;
    return s;
}

// Brackets one launch with events when profiling is on; counts it either way.
struct Timed {
    ptycho_ctx* c; int cls; cudaEvent_t a = nullptr, b = nullptr;
    Timed(ptycho_ctx* c_, int cls_) : c(c_), cls(cls_) {
        if (c->prof) { cudaEventCreate(&a); cudaEventCreate(&b); cudaEventRecord(a, c->stream); }
    }
    ~Timed() {
        ++c->launches;
        if (c->prof) { cudaEventRecord(b, c->stream); c->prof_ev.push_back({cls, a, b}); }
    }
};
#define LAUNCH(c, cls, ...) do { Timed t_(c, cls); __VA_ARGS__; } while (0)

// Frame-size dispatch.  A development build may compile ONE size only (-DPTYCHO_ONLY_N=256: a quarter of the build
// time); the product build (PTYCHO_ONLY_N undefined or 0) instantiates all four.
#ifndef PTYCHO_ONLY_N
#define PTYCHO_ONLY_N 0
#endif
#define PTYCHO_HAS_N(n) (PTYCHO_ONLY_N == 0 || PTYCHO_ONLY_N == (n))
template <int V> struct IntC { static constexpr int value = V; };
template <class F> void dispatch_n(int n, F&& f) {
    switch (n) {
#if PTYCHO_HAS_N(64)
        case 64: f(IntC<64>{}); break;
#endif
#if PTYCHO_HAS_N(128)
        case 128: f(IntC<128>{}); break;
#endif
#if PTYCHO_HAS_N(256)
        case 256: f(IntC<256>{}); break;
#endif
#if PTYCHO_HAS_N(512)
        case 512: f(IntC<512>{}); break;
#endif
        default: break;
    }
}
bool valid_n(int n) { return (n == 64 || n == 128 || n == 256 || n == 512) && PTYCHO_HAS_N(n); }

// Frames per launch of the three-pass kernels (and per piece of fetch / set).  Measured at config 3 (K = 3, batches of 512 frames):
// launches small enough for S to stay in L2 (64 MB: 42 frames, 2.3 waves of CTAs) lose more to their tails than they gain from
// L2 -- 69 ms of kernel time per iteration at 64 MB, 57 at 256 MB, 49 with the whole batch in one launch.  So: a whole minibatch
// per launch, up to 1 GB of scratch.
int chunk_frames(int n, int K, int J, int batch) {
    double mb = 1024.0;
    if (const char* e = getenv("PTYCHO_CHUNK_MB")) mb = atof(e) > 0 ? atof(e) : mb;
    long long per = (long long)K * n * n * 8;
    long long c = std::min<long long>((long long)(mb * 1048576.0) / per, 32768);   // (frames ride in gridDim.y)
    if (batch > 0) c = std::min<long long>(c, batch);
    return (int)std::max<long long>(1, std::min<long long>(c, J));
}

// The only environment switches of the library: the queue geometry of the DM megakernel (PTYCHO_MEGA_M / _D / _X / _RING_MB) and
// the chunk size of the three-pass kernels (PTYCHO_CHUNK_MB).  They change scheduling, never results (tests/test_gpu_parity.py:
// test_dm_queue_geometry_does_not_change_the_result, test_handoff_stress_deterministic_bitwise).
int env_int(const char* name, int dflt) {
    const char* e = getenv(name);
    return (e && *e) ? atoi(e) : dflt;
}
// DM megakernel parameters (single-mode DM only): M frames per wave, D waves of lag, ring R.
int ncb_of(int n);
// Queue geometry.  About grid / (3 NCB) queue waves are in flight at once; a pass-2 item must find its
// pass-1 items finished, a pass-3 item its pass-2 items, and a pass-1 item the ring slot it overwrites
// released, so the lag D and the ring slack X are a little more than that number (measured on cfg2:
// D = X = 8 against D = 4, X = 0 is 9.3 ms against 12.4 ms), and M shrinks until the ring fits the L2 share.
void mega_config(ptycho_ctx* c) {
    c->mega_M = c->mega_D = c->mega_R = 0;
    if (c->K != 1 || c->par.disable_dm || c->par.subpixel_yx) return;   // (sub-pixel positions: per-frame probes, three-pass kernels)
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) { int v = 0; if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0) sms = v; }
    cudaGetLastError();
    const int grid = sms * (c->N >= 512 ? 1 : PTYCHO_MEGA_OCC);
    // About grid / (3 NCB) queue waves are in flight (3 NCB items per wave, + 1 in the split form).
    // Measured on config 2 (B200, round 2): D = 6, X = 5, M = 6 (ring 144 frames, 75 MB) 8.03 / 5.10 ms per early / steady-state
    // iteration (D = 8, X = 7: 8.4 / 5.4); with the earlier sixteen-item pass 2b: M = 6 7.95 / 6.03, M = 3 8.33 / 6.73, M = 2 8.9 / 7.4.  More slots per item amortise the item's probe rows, its claim and
    // its probe-sum flush.
    const int inflight = grid / (3 * ncb_of(c->N) + 1);
    c->mega_D = std::max(2, env_int("PTYCHO_MEGA_D", std::max(3, inflight)));
    const int X = std::max(0, env_int("PTYCHO_MEGA_X", std::max(2, inflight - 1)));
    int M = std::max(1, std::min(env_int("PTYCHO_MEGA_M", 6), c->J));
    // The split form of the queue (dm_mega.cuh) puts three lags between pass 1 and pass 3 of a frame, so the ring spans 3 D + 1 + X
    // waves.  The cap keeps it below the 126 MB L2; next to the streamed exit waves it is nevertheless written back once per
    // iteration (profiles/r02.md: 1.57 x the algorithmic DRAM bytes; a 48 MB ring avoids that and is 0.4-0.7 ms slower).
    const double ring_mb = env_int("PTYCHO_MEGA_RING_MB", 96);
    while (M > 1 && (double)(3 * c->mega_D + 1 + X) * M * c->N * c->N * 8.0 > ring_mb * 1048576.0) --M;
    c->mega_M = M;
    c->mega_R = (3 * c->mega_D + 1 + X) * M;
}

size_t cols_smem(int n, int K) {
    size_t r = 0;
    dispatch_n(n, [&](auto nn) { r = Geo<decltype(nn)::value>::smem_cols(K); });
    return r;
}
int ncb_of(int n) { return n == 64 ? Geo<64>::NCB : n == 128 ? Geo<128>::NCB : n == 256 ? Geo<256>::NCB : Geo<512>::NCB; }

// Lays the workspace out; with base == nullptr only measures it.
size_t layout(ptycho_ctx* c, void* base, bool copy_I) {
    Carver w(base);
    const size_t HW = (size_t)c->H * c->W, nn = (size_t)c->N * c->N, knn = nn * c->K;
    c->O = w.take<float2>(HW);
    const bool want_corr = c->mega_M > 0 && !c->par.deterministic;   // object canvas = correction term, d_O gathered (dm_det.cuh)
    c->p2 = want_corr ? w.take<float>(nn) : nullptr;
    c->dm_stat = w.take<int>(2);
    c->P = w.take<float2>(knn);
    c->nO = w.take<float2>(HW);
    c->dO = w.take<float>(HW);
    c->nP = w.take<float2>(knn);
    c->dP = w.take<float>(nn);
    c->wO = w.take<float>(HW);
    c->pf_part = w.take<double>((size_t)c->J * ncb_of(c->N) * 5);
    c->pf_ab = w.take<float2>(c->J);
    c->S = w.take<float2>((size_t)std::max(c->chunk, c->mega_R) * knn);
    c->mega_ctr = w.take<int>(64 + 4 * (size_t)c->J);
    c->e_part = w.take<float>((size_t)c->J * ncb_of(c->N));
    c->e_tmp = w.take<float>((size_t)c->J * ncb_of(c->N));
    c->tw = w.take<float2>(c->N);
    c->twi = w.take<float2>(c->N);
    c->pos = w.take<YX>(c->J);
    c->spos = w.take<YX>(c->J);
    c->dm_frames = w.take<int>(c->J);
    c->mb_frames = w.take<int>(c->J);
    c->tmp_idx = w.take<int>(c->J);
    c->slot_of = w.take<int>(c->J);
    c->sc = w.take<Scalars>(1);
    c->err_hist = w.take<double>(kErrCap);
    c->steps = w.take<double>(2 * (size_t)kStepCap);
    c->partO = w.take<double>(2 * kRedBlocks);
    c->partP = w.take<double>(2 * kRedBlocks);
    c->partX = w.take<double>((size_t)c->J * kCrossParts);
    c->lsqT = w.take<float2>(nn);
    c->scratch_d = w.take<double>(kRedBlocks);
    c->err_part = w.take<double>(kErrBlocks);
    c->err_ticket = w.take<unsigned int>(1);
    if (!c->par.disable_dm) c->psi = w.take<float2>((size_t)c->J * knn);
    c->It = w.take<char>((size_t)c->J * nn * (c->itype == PTYCHO_I_U16 ? 2 : 4));
    if (c->par.deterministic || want_corr) {                 // frames per object tile: deterministic mode, and the d_O gather
        c->det_tx = (c->W + kDetTileW - 1) / kDetTileW; c->det_ty = (c->H + kDetTileH - 1) / kDetTileH;
        c->tile_start = w.take<int>((size_t)c->det_tx * c->det_ty + 1);
        c->tile_mid = w.take<int>((size_t)c->det_tx * c->det_ty);
        c->tile_list = w.take<int>((size_t)(c->J + c->par.n_foreign) * (c->N / kDetTileW + 1) * (c->N / kDetTileH + 1));   // upper bound
        if (c->par.deterministic || c->par.dm_sweeps > 0) c->det_partial = w.take<float4>((size_t)kDetGroups * nn);
        if (c->par.dm_sweeps > 0) c->tile_slots = w.take<int>((size_t)c->J * (c->N / kDetTileW + 1) * (c->N / kDetTileH + 1));
    }
    // Intensities passed from host memory are needed on the device only during init (sum, re-tiling): they are staged in the
    // exit-wave store, which is not written before the first DM iteration; only without that store do they get their own piece.
    if (c->par.subpixel_yx || !c->sub_frac_h.empty()) {
        c->sub_frac = w.take<float>(2 * (size_t)c->J);
        c->sub_FP = w.take<float2>(knn);
        c->sub_nPF = w.take<float2>(knn);
        c->sub_Pj = w.take<float2>((size_t)c->chunk * knn);
        c->sub_FdP = w.take<float2>(knn);
        c->sub_dPj = w.take<float2>((size_t)c->chunk * knn);
        c->partA22 = w.take<double>((size_t)c->J * kCrossParts);
    }
    if (c->streaming) {
        c->stage_frames = std::max(1, std::min(c->J, (int)((64ull << 20) / (nn * (c->itype == PTYCHO_I_U16 ? 2 : 4)))));
        c->stage = w.take<char>((size_t)c->stage_frames * nn * (c->itype == PTYCHO_I_U16 ? 2 : 4));
        c->scratch_s = w.take<double>(kRedBlocks);
    }
    if (copy_I && !c->streaming) c->I = !c->par.disable_dm ? reinterpret_cast<const void*>(c->psi) : w.take<char>((size_t)c->J * nn * (c->itype == PTYCHO_I_U16 ? 2 : 4));
    return (w.off + 255) & ~size_t(255);
}

bool is_device_ptr(const void* p) {
    cudaPointerAttributes at{};
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

template <int N> ptycho_status set_attrs(ptycho_ctx* c) {
    const int rows = (int)Geo<N>::smem_rows, cols = (int)Geo<N>::smem_cols(c->K);
    if (cols > 227 * 1024) return fail(c, PTYCHO_EUNSUPPORTED, "too many probe modes for this frame size (column-pass staging exceeds shared memory)");
    CU(cudaFuncSetAttribute(k_rows_fwd<N, RF_EXIT>, cudaFuncAttributeMaxDynamicSharedMemorySize, rows));
    CU(cudaFuncSetAttribute(k_rows_fwd<N, RF_DM>, cudaFuncAttributeMaxDynamicSharedMemorySize, rows));
    CU(cudaFuncSetAttribute(k_rows_fwd<N, RF_PLAIN>, cudaFuncAttributeMaxDynamicSharedMemorySize, rows));
    CU(cudaFuncSetAttribute(k_rows_fwd<N, RF_EXIT_PJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, rows));
    CU(cudaFuncSetAttribute(k_rows_fwd<N, RF_DM_PJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, rows));
    CU(cudaFuncSetAttribute(k_rows_inv<N, RI_DM_PJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, rows));
    CU(cudaFuncSetAttribute(k_rows_inv<N, RI_MINIBATCH_PJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, rows));
    CU(cudaFuncSetAttribute(k_rows_inv<N, RI_MINIBATCH>, cudaFuncAttributeMaxDynamicSharedMemorySize, rows));
    CU(cudaFuncSetAttribute(k_rows_inv<N, RI_DM>, cudaFuncAttributeMaxDynamicSharedMemorySize, rows));
    CU(cudaFuncSetAttribute(k_rows_inv<N, RI_REVISED>, cudaFuncAttributeMaxDynamicSharedMemorySize, rows));
    CU(cudaFuncSetAttribute(k_rows_inv<N, RI_PLAIN>, cudaFuncAttributeMaxDynamicSharedMemorySize, rows));
    CU(cudaFuncSetAttribute(k_rows_inv<N, RI_LSQ_PF>, cudaFuncAttributeMaxDynamicSharedMemorySize, rows));
    CU(cudaFuncSetAttribute(k_cols<N, CM_FULL>, cudaFuncAttributeMaxDynamicSharedMemorySize, cols));
    CU(cudaFuncSetAttribute(k_cols<N, CM_ERRONLY>, cudaFuncAttributeMaxDynamicSharedMemorySize, cols));
    CU(cudaFuncSetAttribute(k_cols<N, CM_PLAIN_FWD>, cudaFuncAttributeMaxDynamicSharedMemorySize, cols));
    CU(cudaFuncSetAttribute(k_cols<N, CM_PLAIN_INV>, cudaFuncAttributeMaxDynamicSharedMemorySize, cols));
    CU(cudaFuncSetAttribute(k_dm_mega<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MegaGeo<N>::smem));
    CU(cudaFuncSetAttribute(k_dm_mega<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MegaGeo<N>::smem));
    int per_sm = 0, dev = 0, sms = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_dm_mega<N, true>, kThreads, MegaGeo<N>::smem));
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    c->mega_grid = std::max(1, per_sm) * sms;
    c->sms = sms;
    return PTYCHO_OK;
}

void host_twiddles(int n, int E, int T, std::vector<float2>& tw, std::vector<float2>& twi) {
    tw.resize(n); twi.resize(n);
    for (int ka = 0; ka < E; ++ka)
        for (int b = 0; b < T; ++b) {
            const double ang = -2.0 * M_PI * (double)b * ka / n;
            const float2 w = make_float2((float)cos(ang), (float)sin(ang));
            tw[ka * T + b] = w;
            twi[b * E + ka] = w;
        }
}

FrameArgs base_args(const ptycho_ctx* c) {
    FrameArgs a{};
    a.O = c->O; a.W = c->W; a.P = c->P; a.K = c->K; a.pos = c->pos; a.S = c->S; a.I = c->I; a.itype = c->itype;
    a.It = c->It; a.slot_of = c->slot_of;
    a.nO = c->nO; a.dO = c->dO; a.nP = c->nP; a.dP = c->dP; a.pbound = c->par.pbound; a.tw = c->tw; a.twi = c->twi;
    return a;
}

// The three passes over one chunk.  fwd/col/inv select the kernel variants.
template <int N> void launch_passes(ptycho_ctx* c, const FrameArgs& a, int nframes, int fwd, int col, int inv) {
    using G = Geo<N>;
    const dim3 grid(G::NCB, nframes), blk(kThreads);
    const size_t sr = G::smem_rows, scs = G::smem_cols(c->K);
    cudaStream_t s = c->stream;
    if (fwd >= 0) LAUNCH(c, PTYCHO_K_ROWS_FWD, {
        if (fwd == RF_EXIT) k_rows_fwd<N, RF_EXIT><<<grid, blk, sr, s>>>(a);
        else if (fwd == RF_DM) k_rows_fwd<N, RF_DM><<<grid, blk, sr, s>>>(a);
        else if (fwd == RF_EXIT_PJ) k_rows_fwd<N, RF_EXIT_PJ><<<grid, blk, sr, s>>>(a);
        else if (fwd == RF_DM_PJ) k_rows_fwd<N, RF_DM_PJ><<<grid, blk, sr, s>>>(a);
        else k_rows_fwd<N, RF_PLAIN><<<grid, blk, sr, s>>>(a);
    });
    if (col >= 0) LAUNCH(c, PTYCHO_K_COLS, {
        if (col == CM_FULL) k_cols<N, CM_FULL><<<grid, blk, scs, s>>>(a);
        else if (col == CM_ERRONLY) k_cols<N, CM_ERRONLY><<<grid, blk, scs, s>>>(a);
        else if (col == CM_PLAIN_FWD) k_cols<N, CM_PLAIN_FWD><<<grid, blk, scs, s>>>(a);
        else k_cols<N, CM_PLAIN_INV><<<grid, blk, scs, s>>>(a);
    });
    if (inv >= 0) LAUNCH(c, PTYCHO_K_ROWS_INV, {
        if (inv == RI_MINIBATCH) k_rows_inv<N, RI_MINIBATCH><<<grid, blk, sr, s>>>(a);
        else if (inv == RI_DM) k_rows_inv<N, RI_DM><<<grid, blk, sr, s>>>(a);
        else if (inv == RI_REVISED) k_rows_inv<N, RI_REVISED><<<grid, blk, sr, s>>>(a);
        else if (inv == RI_LSQ_PF) k_rows_inv<N, RI_LSQ_PF><<<grid, blk, sr, s>>>(a);
        else if (inv == RI_MINIBATCH_PJ) k_rows_inv<N, RI_MINIBATCH_PJ><<<grid, blk, sr, s>>>(a);
        else if (inv == RI_DM_PJ) k_rows_inv<N, RI_DM_PJ><<<grid, blk, sr, s>>>(a);
        else k_rows_inv<N, RI_PLAIN><<<grid, blk, sr, s>>>(a);
    });
}

void passes(ptycho_ctx* c, const FrameArgs& a, int nframes, int fwd, int col, int inv) {
    dispatch_n(c->N, [&](auto nn) { launch_passes<decltype(nn)::value>(c, a, nframes, fwd, col, inv); });
}

int ew_blocks(size_t n) { return (int)std::min<size_t>(kRedBlocks, (n + 255) / 256); }

// spatial order (H6): tiles of N/2 rows, boustrophedon in x, so that consecutive frames overlap
void spatial_sort(std::vector<int>& idx, const int32_t* pos, int n) {
    const int tile = std::max(1, n / 2);
    std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) {
        const int ra = pos[2 * a] / tile, rb = pos[2 * b] / tile;
        if (ra != rb) return ra < rb;
        const int xa = pos[2 * a + 1], xb = pos[2 * b + 1];
        return (ra & 1) ? xa > xb : xa < xb;
    });
}

// Minibatch composition (R8) over the frames present, [0, np): strided batches, or runs of the caller's permutation restricted to
// them; every batch spatially sorted.  Rebuilt when more frames have arrived (streaming).
ptycho_status build_batches(ptycho_ctx* c, int np) {
    if (c->mb_built_for == np) return PTYCHO_OK;
    std::vector<int>& mb = c->mb_h;
    if (np < c->J && c->mb_built_for >= 0) CU(cudaStreamSynchronize(c->stream));   // the previous list may still be in flight
    mb.clear();
    c->mb_offsets.assign(1, 0);
    const int B = c->par.batch_size;
    const int32_t* pos = c->pos_h.data();
    if (B <= 0 || B >= np) {
        for (int f : c->dm_order) if (f < np) mb.push_back(f);
        c->mb_offsets.push_back(np);
    } else if (!c->batch_order_h.empty()) {
        std::vector<int> ord;
        for (int f : c->batch_order_h) if (f < np) ord.push_back(f);
        for (int s0 = 0; s0 < np; s0 += B) {
            std::vector<int> fr(ord.begin() + s0, ord.begin() + std::min(np, s0 + B));
            spatial_sort(fr, pos, c->N);
            mb.insert(mb.end(), fr.begin(), fr.end());
            c->mb_offsets.push_back((int)mb.size());
        }
    } else {
        const int nb = (np + B - 1) / B;
        for (int b = 0; b < nb; ++b) {
            std::vector<int> fr;
            for (int j = b; j < np; j += nb) fr.push_back(j);
            spatial_sort(fr, pos, c->N);
            mb.insert(mb.end(), fr.begin(), fr.end());
            c->mb_offsets.push_back((int)mb.size());
        }
    }
    CU(cudaMemcpyAsync(c->mb_frames, mb.data(), (size_t)np * 4, cudaMemcpyHostToDevice, c->stream));
    c->mb_built_for = np;
    return PTYCHO_OK;
}

// Unscaled batched 2-D FFT of `count` N x N frames in place (the plain variants of the three-pass kernels).
void plain_fft2(ptycho_ctx* c, float2* buf, int count, bool inverse) {
    const size_t nn = (size_t)c->N * c->N;
    for (int f0 = 0; f0 < count; f0 += 32768) {             // frames ride in gridDim.y
        FrameArgs a = base_args(c);
        a.S = buf + (size_t)f0 * nn; a.K = 1;
        if (!inverse) passes(c, a, std::min(32768, count - f0), RF_PLAIN, CM_PLAIN_FWD, -1);
        else passes(c, a, std::min(32768, count - f0), -1, CM_PLAIN_INV, RI_PLAIN);
    }
}

// phase: 1 = up to the overlap sums (a1-a9), 2 = the normalising updates (a10), 3 = both.  A shard of a multi-GPU scan runs the
// two halves separately (ptycho_shard_begin / _end) so that the caller can add the other shards' sums in between.
ptycho_status dm_iteration(ptycho_ctx* c, int phase = 3) {
    const size_t nn = (size_t)c->N * c->N, knn = nn * c->K, HW = (size_t)c->H * c->W;
    const int ncb = ncb_of(c->N);
    // R4: psi_j = P O_j before the first DM iteration.  The plain megakernel forms it on the fly in pass 1 (saves a
    // 5 GB write and read at config 2); the other forms of the cycle read the store, so it is written first.
    const bool fresh = !c->psi_valid;
    const bool fresh_in_kernel = fresh && c->mega_M > 0 && !c->par.deterministic;
    if (fresh && !fresh_in_kernel && !c->sub_frac) {
        const dim3 g(c->J, (unsigned)((knn + 255) / 256));   // frame index in grid.x: J may exceed 65535
        LAUNCH(c, PTYCHO_K_OTHER, (k_init_psi<<<g, 256, 0, c->stream>>>(c->psi, c->O, c->W, c->P, c->K, c->N, c->pos, c->dm_frames)));
    }
    const int upd = c->t >= c->par.probe_start;
    if (!(phase & 1)) goto updates;
    if (c->mega_M > 0) {
        MegaArgs m{};
        m.f = base_args(c);
        m.f.psi = c->psi; m.f.frames = c->dm_frames; m.f.e_part = c->e_part;
        m.J = c->J; m.M = c->mega_M; m.D = c->mega_D; m.R = c->mega_R; m.nW = (c->J + m.M - 1) / m.M;
        const int det = c->par.deterministic;
        const int seq = c->par.dm_sweeps;                   // > 0: textbook sequential overlap projection
        m.update_probe = (det || seq) ? 0 : upd;
        m.det = det;
        m.corr = c->p2 ? 1 : 0;
        m.fresh = fresh_in_kernel ? 1 : 0;
        if (det && upd) {                                   // lagged probe sums from the incoming psi (R4), fixed order
            LAUNCH(c, PTYCHO_K_OTHER, (k_det_probe<<<dim3((unsigned)((nn + 255) / 256), kDetGroups), 256, 0, c->stream>>>(
                                           c->det_partial, c->psi, c->O, c->W, c->N, c->spos, c->J)));
            LAUNCH(c, PTYCHO_K_OTHER, (k_det_probe_final<<<(unsigned)((nn + 255) / 256), 256, 0, c->stream>>>(c->nP, c->dP, c->det_partial, (int)nn, kDetGroups)));
        }
        m.spos = c->spos;
        m.It = c->It;
#ifdef PTYCHO_DEBUG
        m.flags = env_int("PTYCHO_MEGA_FLAGS", 0);          // experiment switches of dm_mega.cuh: debug builds only
#else
        m.flags = 0;
#endif
        m.pf = m.M;
        m.head = c->mega_ctr; m.cnt1 = c->mega_ctr + 64; m.cnt2 = m.cnt1 + c->J; m.cnt3 = m.cnt2 + c->J; m.cnt2a = m.cnt3 + c->J;
        m.stat = c->dm_stat;
        if (fresh) CU(cudaMemsetAsync(c->dm_stat, 0, 2 * sizeof(int), c->stream));   // first iteration: fused form
        CU(cudaMemsetAsync(c->mega_ctr, 0, sizeof(int) * (64 + 4 * (size_t)c->J), c->stream));
        {
        const long long items = (long long)(m.nW + 2 * m.D) * 3 * ncb;   // (fused form; the split form has more)
        const int grid = (int)std::min<long long>(items, c->mega_grid);
        const bool u16 = c->itype == PTYCHO_I_U16;
        LAUNCH(c, PTYCHO_K_MEGA, {
            dispatch_n(c->N, [&](auto nn) {
                constexpr int N = decltype(nn)::value;
                if (u16) k_dm_mega<N, true><<<grid, kThreads, MegaGeo<N>::smem, c->stream>>>(m);
                else k_dm_mega<N, false><<<grid, kThreads, MegaGeo<N>::smem, c->stream>>>(m);
            });
        });
        }
    } else if (c->sub_frac) {
        // Sub-pixel positions (R28): per launch the frames' shifted probes; the lagged probe terms conj(O_j) psi_jk stay per frame
        // (sub_dPj), are transformed, multiplied by conj(ramp_j) and summed in Fourier space; one inverse transform gives n_P.
        const float inv_n2 = 1.0f / ((float)c->N * (float)c->N);
        CU(cudaMemcpyAsync(c->sub_FP, c->P, knn * 8, cudaMemcpyDeviceToDevice, c->stream));
        plain_fft2(c, c->sub_FP, c->K, false);
        CU(cudaMemsetAsync(c->sub_nPF, 0, knn * 8, c->stream));
        for (int s0 = 0; s0 < c->J; s0 += c->chunk) {
            const int nf = std::min(c->chunk, c->J - s0);
            const dim3 gr(nf, (unsigned)((knn + 255) / 256));
            LAUNCH(c, PTYCHO_K_OTHER, (k_sub_ramp<<<gr, 256, 0, c->stream>>>(c->sub_Pj, c->sub_FP, c->sub_frac, c->dm_frames + s0, c->K, c->N, inv_n2)));
            plain_fft2(c, c->sub_Pj, nf * c->K, true);
            if (fresh) LAUNCH(c, PTYCHO_K_OTHER, (k_init_psi_pj<<<gr, 256, 0, c->stream>>>(c->psi + (size_t)s0 * knn, c->O, c->W, c->sub_Pj, c->K, c->N, c->pos, c->dm_frames + s0)));
            FrameArgs a = base_args(c);
            a.psi = c->psi + (size_t)s0 * knn;
            a.frames = c->dm_frames + s0;
            a.e_part = c->e_part + (size_t)s0 * ncb;
            a.Pj = c->sub_Pj; a.Gj = c->sub_dPj;
            passes(c, a, nf, RF_DM_PJ, CM_FULL, RI_DM_PJ);
            plain_fft2(c, c->sub_dPj, nf * c->K, false);
            LAUNCH(c, PTYCHO_K_OTHER, (k_sub_acc<<<(unsigned)((knn + 255) / 256), 256, 0, c->stream>>>(c->sub_nPF, c->sub_dPj, c->sub_frac, c->dm_frames + s0, nf, c->K, c->N)));
        }
        plain_fft2(c, c->sub_nPF, c->K, true);
        LAUNCH(c, PTYCHO_K_OTHER, (k_scale_to<<<ew_blocks(knn), 256, 0, c->stream>>>(c->nP, c->sub_nPF, knn, inv_n2)));
    } else
    for (int s0 = 0; s0 < c->J; s0 += c->chunk) {
        const int nf = std::min(c->chunk, c->J - s0);
        FrameArgs a = base_args(c);
        a.psi = c->psi + (size_t)s0 * knn;
        a.frames = c->dm_frames + s0;
        a.e_part = c->e_part + (size_t)s0 * ncb;
        passes(c, a, nf, RF_DM, CM_FULL, RI_DM);
    }
    c->psi_valid = true;                                    // (a failed launch returns above)
    if (!(phase & 2)) { CU(cudaGetLastError()); return PTYCHO_OK; }
updates:
    if (c->par.deterministic)                               // object sums from the new psi, fixed order
        LAUNCH(c, PTYCHO_K_OTHER, (k_det_object<<<dim3(c->det_tx, c->det_ty), dim3(kDetTileW, kDetTileH), 0, c->stream>>>(
                                       c->nO, c->dO, c->H, c->W, c->psi, c->P, c->N, c->spos, c->tile_start, c->tile_list)));
    if (c->mega_M > 0 && c->p2) {                           // O += c / (d_O + eps), d_O gathered over the tile lists (dm_det.cuh)
        LAUNCH(c, PTYCHO_K_UPDATE, (k_probe_support<<<(unsigned)((nn + 1023) / 1024), 1024, 0, c->stream>>>(c->p2, c->P, c->N, c->dm_stat)));
        LAUNCH(c, PTYCHO_K_UPDATE, (k_dm_blend_gather<<<dim3(c->det_tx, c->det_ty), dim3(kDetTileW, kDetTileH), 0, c->stream>>>(
                                        c->O, c->nO, c->H, c->W, c->p2, c->N, c->tile_start, c->tile_mid, c->tile_list, c->sc)));
    }
    else
        LAUNCH(c, PTYCHO_K_UPDATE, (k_dm_blend<<<ew_blocks(HW), 256, 0, c->stream>>>(c->O, c->nO, c->dO, HW, 1, c->sc, 0, 1)));
    if (c->par.dm_sweeps > 0 && c->mega_M > 0) {
        // sequential form: the object above came from the new exit waves with the old probe; now the probe from the same waves
        // and the NEW object (fixed-order gathers of dm_det.cuh), then further object / probe sweeps.
        for (int sw = 0; sw < c->par.dm_sweeps; ++sw) {
            if (sw > 0) {
                LAUNCH(c, PTYCHO_K_OTHER, (k_det_object<<<dim3(c->det_tx, c->det_ty), dim3(kDetTileW, kDetTileH), 0, c->stream>>>(
                                               c->nO, c->dO, c->H, c->W, c->psi, c->P, c->N, c->spos, c->tile_start, c->tile_slots)));
                LAUNCH(c, PTYCHO_K_UPDATE, (k_dm_blend<<<ew_blocks(HW), 256, 0, c->stream>>>(c->O, c->nO, c->dO, HW, 1, c->sc, 0, 1)));
            }
            if (upd) {
                LAUNCH(c, PTYCHO_K_OTHER, (k_det_probe<<<dim3((unsigned)((nn + 255) / 256), kDetGroups), 256, 0, c->stream>>>(
                                               c->det_partial, c->psi, c->O, c->W, c->N, c->spos, c->J)));
                LAUNCH(c, PTYCHO_K_OTHER, (k_det_probe_final<<<(unsigned)((nn + 255) / 256), 256, 0, c->stream>>>(c->nP, c->dP, c->det_partial, (int)nn, kDetGroups)));
                LAUNCH(c, PTYCHO_K_UPDATE, (k_dm_blend<<<ew_blocks(nn), 256, 0, c->stream>>>(c->P, c->nP, c->dP, nn, c->K, c->sc, 1, 1)));
            }
        }
    } else
        LAUNCH(c, PTYCHO_K_UPDATE, (k_dm_blend<<<ew_blocks(nn), 256, 0, c->stream>>>(c->P, c->nP, c->dP, nn, c->K, c->sc, 1, upd)));
    CU(cudaGetLastError());
    c->psi_valid = true;                                    // only once every launch of the iteration has been accepted
    return PTYCHO_OK;
}

ptycho_status minibatch_iteration(ptycho_ctx* c, ptycho_alg alg) {
    const size_t nn = (size_t)c->N * c->N, HW = (size_t)c->H * c->W;
    const int ncb = ncb_of(c->N);
    const int upd = c->t >= c->par.probe_start;
    const int nb = (int)c->mb_offsets.size() - 1;
    for (int b = 0; b < nb; ++b) {
        const int b0 = c->mb_offsets[b], b1 = c->mb_offsets[b + 1];
        const bool epie = alg == PTYCHO_EPIE_MB;
        if (!epie) c->epie_pi = -1;
        if (!epie || c->epie_pi < 0) {                      // (ePIE: the previous batch's probe update left the maximum behind)
            CU(cudaMemsetAsync(&c->sc->max_p2, 0, sizeof(float), c->stream));
            LAUNCH(c, PTYCHO_K_UPDATE, (k_probe_max<<<64, 256, 0, c->stream>>>(c->P, c->K, (int)nn, c->sc)));
        }
        if (c->sub_frac) {
            // Sub-pixel positions (R28).  Per launch: the frames' shifted probes P_jk = F^-1[F[P_k] ramp_j] into sub_Pj, the cycle with
            // them (the inverse row pass leaves the probe terms conj(O_j) chi_jk in sub_Pj), their spectra times conj(ramp_j) summed
            // into sub_nPF; per batch one inverse transform brings the sum back: n_P = F^-1[sub_nPF].
            const size_t knn = nn * c->K;
            const float inv_n2 = 1.0f / ((float)c->N * (float)c->N);
            CU(cudaMemcpyAsync(c->sub_FP, c->P, knn * 8, cudaMemcpyDeviceToDevice, c->stream));
            plain_fft2(c, c->sub_FP, c->K, false);
            CU(cudaMemsetAsync(c->sub_nPF, 0, knn * 8, c->stream));
            for (int s0 = b0; s0 < b1; s0 += c->chunk) {
                const int nf = std::min(c->chunk, b1 - s0);
                LAUNCH(c, PTYCHO_K_OTHER, (k_sub_ramp<<<dim3(nf, (unsigned)((knn + 255) / 256)), 256, 0, c->stream>>>(
                                               c->sub_Pj, c->sub_FP, c->sub_frac, c->mb_frames + s0, c->K, c->N, inv_n2)));
                plain_fft2(c, c->sub_Pj, nf * c->K, true);
                FrameArgs a = base_args(c);
                a.frames = c->mb_frames + s0;
                a.e_part = c->e_part + (size_t)s0 * ncb;
                a.Pj = c->sub_Pj;
                passes(c, a, nf, RF_EXIT_PJ, CM_FULL, RI_MINIBATCH_PJ);
                plain_fft2(c, c->sub_Pj, nf * c->K, false);
                LAUNCH(c, PTYCHO_K_OTHER, (k_sub_acc<<<(unsigned)((knn + 255) / 256), 256, 0, c->stream>>>(
                                               c->sub_nPF, c->sub_Pj, c->sub_frac, c->mb_frames + s0, nf, c->K, c->N)));
            }
            plain_fft2(c, c->sub_nPF, c->K, true);
            LAUNCH(c, PTYCHO_K_OTHER, (k_scale_to<<<ew_blocks(knn), 256, 0, c->stream>>>(c->nP, c->sub_nPF, knn, inv_n2)));
        } else
        for (int s0 = b0; s0 < b1; s0 += c->chunk) {
            const int nf = std::min(c->chunk, b1 - s0);
            FrameArgs a = base_args(c);
            a.frames = c->mb_frames + s0;
            a.e_part = c->e_part + (size_t)s0 * ncb;
            passes(c, a, nf, RF_EXIT, CM_FULL, RI_MINIBATCH);
        }
        const bool lsq = alg == PTYCHO_LSQML, pfm = alg == PTYCHO_LSQML_PF;
        const int gO = ew_blocks(HW), gP = ew_blocks(nn);
        if (!lsq && !pfm) {                                 // ePIE: directions and steps in one pass per canvas
            const int pi = c->epie_pi, pw = pi < 0 ? 0 : 1 - pi;
            LAUNCH(c, PTYCHO_K_UPDATE, (k_epie_update<<<gO, 256, 0, c->stream>>>(c->O, c->nO, c->dO, HW, 1, c->par.delta_obj, c->par.alpha_obj, c->sc, 0, 1,
                                                                                 pi, pw, nullptr, 0.f, 0.f)));   // (zeroes max_dp and max_p2s[pw])
            if (upd) LAUNCH(c, PTYCHO_K_UPDATE, (k_real_max<<<64, 256, 0, c->stream>>>(c->dP, (int)nn, c->sc)));
            LAUNCH(c, PTYCHO_K_UPDATE, (k_epie_update<<<gP, 256, 0, c->stream>>>(c->P, c->nP, c->dP, nn, c->K, c->par.delta_probe, c->par.alpha_probe, c->sc, 1, upd,
                                                                                 -1, pw, c->n_steps < kStepCap ? c->steps + 2 * c->n_steps : nullptr,
                                                                                 c->par.alpha_obj, upd ? c->par.alpha_probe : 0.f)));
            c->epie_pi = pw;
            ++c->n_steps;
            continue;
        }
        LAUNCH(c, PTYCHO_K_UPDATE, (k_direction<<<gO, 256, 0, c->stream>>>(c->nO, c->dO, HW, 1, c->par.delta_obj, c->sc, 0, lsq ? c->partO : nullptr)));
        if (upd) {
            CU(cudaMemsetAsync(&c->sc->max_dp, 0, sizeof(float), c->stream));
            LAUNCH(c, PTYCHO_K_UPDATE, (k_real_max<<<64, 256, 0, c->stream>>>(c->dP, (int)nn, c->sc)));
            LAUNCH(c, PTYCHO_K_UPDATE, (k_direction<<<gP, 256, 0, c->stream>>>(c->nP, c->dP, nn, c->K, c->par.delta_probe, c->sc, 1, lsq ? c->partP : nullptr)));
        }
        double* step_slot = c->n_steps < kStepCap ? c->steps + 2 * c->n_steps : nullptr;
        if (pfm) {
            // R25: a second transform cycle over the batch recomputes chi_j and leaves every frame's five sums; then the per-frame
            // solves, the weighted second scatter (a_j w_j into dO, which the directions no longer need; w_j into wO) and the updates.
            for (int s0 = b0; s0 < b1; s0 += c->chunk) {
                const int nf = std::min(c->chunk, b1 - s0);
                FrameArgs a = base_args(c);
                a.frames = c->mb_frames + s0;
                a.e_part = c->e_part + (size_t)s0 * ncb;
                a.pf_part = c->pf_part + (size_t)(s0 - b0) * ncb * 5;
                passes(c, a, nf, RF_EXIT, CM_FULL, RI_LSQ_PF);
            }
            const int cap = (int)std::max<long long>(0, std::min<long long>(b1 - b0, kStepCap - c->n_steps));
            LAUNCH(c, PTYCHO_K_UPDATE, (k_lsq_pf_solve<<<1, 1024, 0, c->stream>>>(c->pf_part, b1 - b0, ncb, c->par.lsq_lambda, upd, c->pf_ab, c->sc,
                                                                               cap > 0 ? c->steps + 2 * c->n_steps : nullptr, cap)));
            CU(cudaMemsetAsync(c->dO, 0, HW * 4, c->stream));
            LAUNCH(c, PTYCHO_K_UPDATE, (k_lsq_pf_scatter<<<dim3(b1 - b0, (unsigned)((nn + 255) / 256)), 256, 0, c->stream>>>(
                                            c->dO, c->wO, c->W, c->P, c->K, c->N, c->pos, c->mb_frames + b0, c->pf_ab)));
            LAUNCH(c, PTYCHO_K_UPDATE, (k_lsq_pf_apply<<<gO, 256, 0, c->stream>>>(c->O, c->nO, c->dO, c->wO, HW)));
            LAUNCH(c, PTYCHO_K_UPDATE, (k_apply<<<gP, 256, 0, c->stream>>>(c->P, c->nP, c->dP, nn, c->K, c->sc, 1, upd)));
            c->n_steps += b1 - b0;
            continue;
        }
        if (lsq && c->sub_frac && upd) {
            // Sub-pixel positions: A22 and A12 from their per-frame definitions (R28).  F[dP] once, then per launch the frames'
            // shifted probes (again: sub_Pj was used up by the cycle) and shifted probe directions, and the per-frame gather.
            const size_t knn = nn * c->K;
            const float inv_n2 = 1.0f / ((float)c->N * (float)c->N);
            const int log2n = c->N == 64 ? 6 : c->N == 128 ? 7 : c->N == 256 ? 8 : 9;
            CU(cudaMemcpyAsync(c->sub_FdP, c->nP, knn * 8, cudaMemcpyDeviceToDevice, c->stream));
            plain_fft2(c, c->sub_FdP, c->K, false);
            for (int s0 = b0; s0 < b1; s0 += c->chunk) {
                const int nf = std::min(c->chunk, b1 - s0);
                const dim3 gr(nf, (unsigned)((knn + 255) / 256));
                LAUNCH(c, PTYCHO_K_OTHER, (k_sub_ramp<<<gr, 256, 0, c->stream>>>(c->sub_Pj, c->sub_FP, c->sub_frac, c->mb_frames + s0, c->K, c->N, inv_n2)));
                LAUNCH(c, PTYCHO_K_OTHER, (k_sub_ramp<<<gr, 256, 0, c->stream>>>(c->sub_dPj, c->sub_FdP, c->sub_frac, c->mb_frames + s0, c->K, c->N, inv_n2)));
                plain_fft2(c, c->sub_Pj, nf * c->K, true);
                plain_fft2(c, c->sub_dPj, nf * c->K, true);
                LAUNCH(c, PTYCHO_K_UPDATE, (k_lsq_cross_pj<<<dim3(nf, kCrossParts), 256, 0, c->stream>>>(
                                                c->O, c->nO, c->W, c->sub_Pj, c->sub_dPj, c->K, c->N, log2n, c->pos, c->mb_frames + s0,
                                                c->partX + (size_t)(s0 - b0) * kCrossParts, c->partA22 + (size_t)(s0 - b0) * kCrossParts)));
            }
            LAUNCH(c, PTYCHO_K_UPDATE, (k_lsq_solve<<<1, 256, 0, c->stream>>>(c->partO, gO, c->partP, gP, c->partX, (b1 - b0) * kCrossParts,
                                                                            c->par.lsq_lambda, upd, c->sc, step_slot ? step_slot : c->scratch_d, c->partA22)));
        } else if (lsq) {
            if (upd) {
                const int log2n = c->N == 64 ? 6 : c->N == 128 ? 7 : c->N == 256 ? 8 : 9;
                LAUNCH(c, PTYCHO_K_UPDATE, (k_lsq_T<<<(unsigned)((nn + 255) / 256), 256, 0, c->stream>>>(c->lsqT, c->P, c->nP, c->K, (int)nn)));
                LAUNCH(c, PTYCHO_K_UPDATE, (k_lsq_cross<<<dim3(b1 - b0, kCrossParts), 256, 0, c->stream>>>(c->O, c->nO, c->W, c->lsqT, c->N, log2n, c->pos,
                                                                                        c->mb_frames + b0, c->partX)));
            }
            LAUNCH(c, PTYCHO_K_UPDATE, (k_lsq_solve<<<1, 256, 0, c->stream>>>(c->partO, gO, c->partP, upd ? gP : 0, c->partX, upd ? (b1 - b0) * kCrossParts : 0,
                                                                            c->par.lsq_lambda, upd, c->sc, step_slot ? step_slot : c->scratch_d)));
        } else {
            LAUNCH(c, PTYCHO_K_UPDATE, (k_set_steps<<<1, 1, 0, c->stream>>>(c->sc, c->par.alpha_obj, upd ? c->par.alpha_probe : 0.f, step_slot)));
        }
        ++c->n_steps;
        LAUNCH(c, PTYCHO_K_UPDATE, (k_apply<<<gO, 256, 0, c->stream>>>(c->O, c->nO, c->dO, HW, 1, c->sc, 0, 1)));
        LAUNCH(c, PTYCHO_K_UPDATE, (k_apply<<<gP, 256, 0, c->stream>>>(c->P, c->nP, c->dP, nn, c->K, c->sc, 1, upd)));
    }
    c->psi_valid = false;
    return PTYCHO_OK;
}

}  // namespace

// =========================================================================================
// C ABI
// =========================================================================================
extern "C" {

void ptycho_default_params(ptycho_params* p) {
    if (!p) return;
    memset(p, 0, sizeof(*p));
    p->delta_blend = 1e-2f;
    p->delta_obj = 1.0f;
    p->delta_probe = 1.0f;
    p->alpha_obj = 1.0f;
    p->alpha_probe = 1.0f;
    p->lsq_lambda = 0.1f;
}

size_t ptycho_workspace_bytes(int obj_h, int obj_w, int n, int n_modes, int n_pos, ptycho_itype itype,
                              int intensities_on_host, const ptycho_params* params) {
    if (!valid_n(n) || n_modes < 1 || n_modes > PTYCHO_MAX_MODES || n_pos < 1 || obj_h < n || obj_w < n) return 0;
    ptycho_ctx tmp;
    tmp.H = obj_h; tmp.W = obj_w; tmp.N = n; tmp.K = n_modes; tmp.J = n_pos; tmp.itype = itype;
    if (params) tmp.par = *params; else ptycho_default_params(&tmp.par);
    tmp.chunk = chunk_frames(n, n_modes, n_pos, tmp.par.batch_size);
    mega_config(&tmp);
    tmp.streaming = intensities_on_host == 2;
    return layout(&tmp, nullptr, intensities_on_host == 1);
}

ptycho_status ptycho_init(ptycho_ctx** out, const float* object, int obj_h, int obj_w, const float* probe,
                          int n_modes, int n, const int32_t* pos_yx, int n_pos, const void* intensities,
                          ptycho_itype itype, const ptycho_params* params, void* workspace, size_t workspace_bytes,
                          void* cuda_stream) {
    ptycho_ctx* c = nullptr;
    if (!out) return PTYCHO_EINVAL;
    *out = nullptr;
    if (!object || !probe || !pos_yx || !workspace) return PTYCHO_EINVAL;   // intensities == NULL: streaming context (ptycho_append_frames)
    if (!valid_n(n) || n_modes < 1 || n_pos < 1 || obj_h < n || obj_w < n) return PTYCHO_EINVAL;
    if (itype != PTYCHO_I_F32 && itype != PTYCHO_I_U16) return PTYCHO_EINVAL;
    if (n_modes > PTYCHO_MAX_MODES) return PTYCHO_EUNSUPPORTED;
    ptycho_params par;
    if (params) par = *params; else ptycho_default_params(&par);
    if (par.batch_size < 0 || par.pbound < 0 || par.delta_blend <= 0 || par.delta_obj <= 0 || par.delta_probe <= 0)
        return PTYCHO_EINVAL;
    // deterministic mode (dm_det.cuh) is built for the single-mode DM megakernel path only
    if (par.deterministic && (n_modes != 1 || par.disable_dm)) return PTYCHO_EUNSUPPORTED;
    if (par.dm_sweeps < 0) return PTYCHO_EINVAL;
    if (par.dm_sweeps > 0 && (n_modes != 1 || par.disable_dm || par.deterministic)) return PTYCHO_EUNSUPPORTED;
    if (cols_smem(n, n_modes) > 227 * 1024) return PTYCHO_EUNSUPPORTED;
    const bool shard = par.shard_total_pos > 0;
    if (par.shard_total_pos < 0 || par.n_foreign < 0 || (par.n_foreign > 0 && !par.foreign_pos)) return PTYCHO_EINVAL;
    if (!shard && par.n_foreign > 0) return PTYCHO_EINVAL;
    if (shard && par.shard_total_pos < n_pos + par.n_foreign) return PTYCHO_EINVAL;
    if (shard && (n_modes != 1 || par.disable_dm || par.deterministic || par.dm_sweeps > 0 || !intensities)) return PTYCHO_EUNSUPPORTED;
    if (par.subpixel_yx) {
        if (par.deterministic || par.dm_sweeps > 0 || shard || !intensities) return PTYCHO_EUNSUPPORTED;
        for (int j = 0; j < 2 * n_pos; ++j)
            if (!(par.subpixel_yx[j] >= 0.f && par.subpixel_yx[j] < 1.f)) return PTYCHO_EINVAL;
    }
    for (int j = 0; j < par.n_foreign; ++j) {
        const int y = par.foreign_pos[2 * j], x = par.foreign_pos[2 * j + 1];
        if (y < 0 || x < 0 || y + n > obj_h || x + n > obj_w) return PTYCHO_EBOUNDS;
    }

    // positions: copy, check bounds (R10), accept host or device memory
    std::vector<int32_t> pos(2 * (size_t)n_pos);
    if (is_device_ptr(pos_yx)) {
        if (cudaMemcpy(pos.data(), pos_yx, pos.size() * 4, cudaMemcpyDeviceToHost) != cudaSuccess) return PTYCHO_ECUDA;
    } else memcpy(pos.data(), pos_yx, pos.size() * 4);
    for (int j = 0; j < n_pos; ++j) {
        const int y = pos[2 * j], x = pos[2 * j + 1];
        if (y < 0 || x < 0 || y + n > obj_h || x + n > obj_w) return PTYCHO_EBOUNDS;
    }
    if (par.batch_order) {                                  // must be a permutation
        std::vector<char> seen(n_pos, 0);
        for (int i = 0; i < n_pos; ++i) {
            const int v = par.batch_order[i];
            if (v < 0 || v >= n_pos || seen[v]) return PTYCHO_EINVAL;
            seen[v] = 1;
        }
    }
    if (!is_device_ptr(workspace)) return PTYCHO_EINVAL;

    c = new ptycho_ctx;
    c->H = obj_h; c->W = obj_w; c->N = n; c->K = n_modes; c->J = n_pos; c->itype = itype; c->par = par;
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    c->chunk = chunk_frames(n, n_modes, n_pos, par.batch_size);
    mega_config(c);
    c->streaming = intensities == nullptr;
    const bool dev_I = c->streaming || is_device_ptr(intensities);
    const size_t need = layout(c, nullptr, !dev_I);
    if (workspace_bytes < need || (reinterpret_cast<uintptr_t>(workspace) & 255)) { delete c; return PTYCHO_ENOMEM; }
    layout(c, workspace, !dev_I);
    if (dev_I) c->I = intensities;
    c->present = c->streaming ? 0 : n_pos;
    if (c->streaming) {
        if (cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) != cudaSuccess || cudaEventCreateWithFlags(&c->ev_append, cudaEventDisableTiming) != cudaSuccess) { delete c; return PTYCHO_ECUDA; }
    }

#define CUI(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { g_init_error = std::string(#call) + ": " + cudaGetErrorString(e_); delete c; return PTYCHO_ECUDA; } } while (0)
    ptycho_status st = PTYCHO_OK;
    dispatch_n(n, [&](auto nn) { st = set_attrs<decltype(nn)::value>(c); });
    if (st != PTYCHO_OK) { g_init_error = c->err; delete c; return st; }

    const size_t HW = (size_t)obj_h * obj_w, nn = (size_t)n * n, knn = nn * n_modes;
    cudaStream_t s = c->stream;
    CUI(cudaMemcpyAsync(c->O, object, HW * 8, cudaMemcpyDefault, s));
    CUI(cudaMemcpyAsync(c->P, probe, knn * 8, cudaMemcpyDefault, s));
    if (!dev_I) CUI(cudaMemcpyAsync(const_cast<void*>(c->I), intensities, (size_t)n_pos * nn * (itype == PTYCHO_I_U16 ? 2 : 4), cudaMemcpyDefault, s));
    CUI(cudaMemcpyAsync(c->pos, pos.data(), pos.size() * 4, cudaMemcpyHostToDevice, s));
    CUI(cudaMemsetAsync(c->nO, 0, HW * 8, s));
    CUI(cudaMemsetAsync(c->dO, 0, HW * 4, s));
    CUI(cudaMemsetAsync(c->nP, 0, knn * 8, s));
    CUI(cudaMemsetAsync(c->dP, 0, nn * 4, s));
    CUI(cudaMemsetAsync(c->wO, 0, HW * 4, s));
    CUI(cudaMemsetAsync(c->sc, 0, sizeof(Scalars), s));
    CUI(cudaMemsetAsync(c->err_hist, 0, sizeof(double) * kErrCap, s));
    CUI(cudaMemsetAsync(c->err_ticket, 0, sizeof(unsigned int), s));
    CUI(cudaMemsetAsync(c->e_part, 0, sizeof(float) * (size_t)n_pos * ncb_of(n), s));
    CUI(cudaMemsetAsync(c->dm_stat, 0, 2 * sizeof(int), s));

    std::vector<float2> tw, twi;
    const int E = n == 64 ? 8 : n == 512 ? 32 : 16, T = n / E;
    host_twiddles(n, E, T, tw, twi);
    CUI(cudaMemcpyAsync(c->tw, tw.data(), n * 8, cudaMemcpyHostToDevice, s));
    CUI(cudaMemcpyAsync(c->twi, twi.data(), n * 8, cudaMemcpyHostToDevice, s));

    // frame orders: DM = all frames, spatially sorted; minibatch = batches (R8), each sorted
    c->dm_order.resize(n_pos);
    std::iota(c->dm_order.begin(), c->dm_order.end(), 0);
    spatial_sort(c->dm_order, pos.data(), n);
    c->slot_of_h.resize(n_pos);
    for (int sidx = 0; sidx < n_pos; ++sidx) c->slot_of_h[c->dm_order[sidx]] = sidx;
    c->pos_h = pos;
    if (par.batch_order) c->batch_order_h.assign(par.batch_order, par.batch_order + n_pos);
    c->par.batch_order = nullptr;   // copied; the caller's pointer is not kept
    if (par.n_foreign > 0) c->foreign_h.assign(par.foreign_pos, par.foreign_pos + 2 * (size_t)par.n_foreign);
    c->par.foreign_pos = nullptr;
    if (par.subpixel_yx) {
        c->sub_frac_h.assign(par.subpixel_yx, par.subpixel_yx + 2 * (size_t)n_pos);
        CUI(cudaMemcpyAsync(c->sub_frac, c->sub_frac_h.data(), c->sub_frac_h.size() * 4, cudaMemcpyHostToDevice, s));
    }
    c->par.subpixel_yx = nullptr;
    if (shard) {
        if (!c->p2) { g_init_error = "a shard needs the DM megakernel path"; delete c; return PTYCHO_EUNSUPPORTED; }
        int r0 = obj_h, r1 = 0;
        for (int j = 0; j < n_pos; ++j) { r0 = std::min(r0, pos[2 * j]); r1 = std::max(r1, pos[2 * j] + n); }
        c->shard_row0 = r0; c->shard_row1 = r1;
    }
    CUI(cudaMemcpyAsync(c->dm_frames, c->dm_order.data(), n_pos * 4, cudaMemcpyHostToDevice, s));
    std::vector<int32_t> spos(2 * (size_t)n_pos);
    for (int sidx = 0; sidx < n_pos; ++sidx) { spos[2 * sidx] = pos[2 * c->dm_order[sidx]]; spos[2 * sidx + 1] = pos[2 * c->dm_order[sidx] + 1]; }
    CUI(cudaMemcpyAsync(c->spos, spos.data(), spos.size() * 4, cudaMemcpyHostToDevice, s));
    CUI(cudaMemcpyAsync(c->slot_of, c->slot_of_h.data(), n_pos * 4, cudaMemcpyHostToDevice, s));

    if (par.deterministic || c->p2) {                       // frames per object tile, ascending slot (dm_det.cuh)
        // deterministic mode: entries are slots.  Otherwise (the d_O gather of k_dm_blend_gather): entries are packed positions
        // y << 16 | x, and the frames that cover the WHOLE tile come first (tile_mid marks the boundary): no per-pixel test for them.
        const bool gather = !par.deterministic;
        const size_t ntiles = (size_t)c->det_tx * c->det_ty;
        std::vector<int> start(ntiles + 1, 0), mid(ntiles, 0), list, slots;
        const bool want_slots = gather && par.dm_sweeps > 0;
        auto whole = [&](int y, int x, int ty, int tx) {
            return y <= ty * kDetTileH && (ty + 1) * kDetTileH <= y + n && x <= tx * kDetTileW && (tx + 1) * kDetTileW <= x + n;
        };
        for (int pass = 0; pass < 2; ++pass) {
            std::vector<int> fill_a, fill_b, fill_s;
            if (pass == 1) {
                fill_a.assign(start.begin(), start.end() - 1);
                fill_b.resize(ntiles);
                for (size_t i = 0; i < ntiles; ++i) { fill_b[i] = start[i] + mid[i]; mid[i] = fill_b[i]; }
                if (want_slots) fill_s.assign(start.begin(), start.end() - 1);
            }
            // a shard also lists the other shards' frames over its rows (they enter d_O only): entries n_pos .. n_pos + n_foreign - 1
            const int n_list = n_pos + (gather ? par.n_foreign : 0);
            for (int sidx = 0; sidx < n_list; ++sidx) {
                const int y = sidx < n_pos ? spos[2 * sidx] : c->foreign_h[2 * (size_t)(sidx - n_pos)];
                const int x = sidx < n_pos ? spos[2 * sidx + 1] : c->foreign_h[2 * (size_t)(sidx - n_pos) + 1];
                for (int ty = y / kDetTileH; ty <= (y + n - 1) / kDetTileH; ++ty)
                    for (int tx = x / kDetTileW; tx <= (x + n - 1) / kDetTileW; ++tx) {
                        const size_t tl = (size_t)ty * c->det_tx + tx;
                        const bool w = gather && whole(y, x, ty, tx);
                        if (pass == 0) { ++start[tl + 1]; if (w) ++mid[tl]; continue; }
                        if (want_slots) slots[fill_s[tl]++] = sidx;
                        if (!gather) list[fill_a[tl]++] = sidx;
                        else if (w) list[fill_a[tl]++] = (y << 16) | x;
                        else list[fill_b[tl]++] = (y << 16) | x;
                    }
            }
            if (pass == 0) { for (size_t i = 0; i < ntiles; ++i) start[i + 1] += start[i]; list.resize(start[ntiles]); if (want_slots) slots.resize(start[ntiles]); }
        }
        if (shard)                                          // one summation order of d_O on every shard that covers a tile: by position
            for (size_t i = 0; i < ntiles; ++i) {
                std::sort(list.begin() + start[i], list.begin() + mid[i]);
                std::sort(list.begin() + mid[i], list.begin() + start[i + 1]);
            }
        if (want_slots) CUI(cudaMemcpyAsync(c->tile_slots, slots.data(), slots.size() * 4, cudaMemcpyHostToDevice, s));
        CUI(cudaMemcpyAsync(c->tile_start, start.data(), start.size() * 4, cudaMemcpyHostToDevice, s));
        CUI(cudaMemcpyAsync(c->tile_mid, mid.data(), mid.size() * 4, cudaMemcpyHostToDevice, s));
        CUI(cudaMemcpyAsync(c->tile_list, list.data(), list.size() * 4, cudaMemcpyHostToDevice, s));
        CUI(cudaStreamSynchronize(s));                      // the host vectors go out of scope
    }
    if (!c->streaming) {                                    // intensities in pass-2 tile order (dm_mega.cuh)
        const dim3 g(n_pos, ncb_of(n));   // frame index in grid.x: J may exceed 65535
#define TILE_I(NN) do { if (itype == PTYCHO_I_U16) k_tile_intensity<NN, unsigned short><<<g, kThreads, 0, s>>>((unsigned short*)c->It, (const unsigned short*)c->I, c->dm_frames); \
                        else k_tile_intensity<NN, float><<<g, kThreads, 0, s>>>((float*)c->It, (const float*)c->I, c->dm_frames); } while (0)
        dispatch_n(n, [&](auto nn) { constexpr int NN = decltype(nn)::value; TILE_I(NN); });
#undef TILE_I
        ++c->launches;
    }
    // init-time constants on the device: eps_O, eps_P (R5), sum_I (C3)
    k_probe_max<<<64, 256, 0, s>>>(c->P, c->K, (int)nn, c->sc);   // sc was zeroed above
    k_finish_init<<<1, 1, 0, s>>>(c->sc, par.delta_blend, n_pos, 0);
    k_abs2_max<<<ew_blocks(HW), 256, 0, s>>>(c->O, HW, c->sc);
    k_finish_init<<<1, 1, 0, s>>>(c->sc, par.delta_blend, shard ? par.shard_total_pos : n_pos, 1);
    if (!c->streaming) {
        k_sum_intensity<<<kRedBlocks, 256, 0, s>>>(c->I, itype, (size_t)n_pos * nn, c->scratch_d);
        k_finish_sum_I<<<1, 32, 0, s>>>(c->scratch_d, kRedBlocks, c->sc, 0);
        c->launches += 2;
    }
    c->launches += 4;
    CUI(cudaStreamSynchronize(s));
    CUI(cudaGetLastError());
#undef CUI
    if ((!dev_I && !c->par.disable_dm) || c->streaming) c->I = nullptr;       // the staging copy lived in the exit-wave store: gone after init
    *out = c;
    return PTYCHO_OK;
}

ptycho_status ptycho_iterate(ptycho_ctx* c, ptycho_alg alg, int n_iters) {
    if (!c || n_iters < 0) return PTYCHO_EINVAL;
    if (alg != PTYCHO_EPIE_MB && alg != PTYCHO_DM && alg != PTYCHO_LSQML && alg != PTYCHO_LSQML_PF) return fail(c, PTYCHO_EINVAL, "unknown algorithm");
    if (alg != PTYCHO_DM && c->par.deterministic) return fail(c, PTYCHO_EUNSUPPORTED, "deterministic mode covers DM only");
    if (alg == PTYCHO_DM && !c->psi) return fail(c, PTYCHO_ESTATE, "DM needs the exit-wave store (disable_dm was set)");
    if (c->par.shard_total_pos > 0) return fail(c, PTYCHO_ESTATE, "a shard is driven by ptycho_shard_begin / ptycho_shard_end");
    if (c->sub_frac && alg == PTYCHO_LSQML_PF) return fail(c, PTYCHO_EUNSUPPORTED, "sub-pixel positions: not with per-frame LSQML steps");
    if (c->streaming) {
        if (c->present == 0) return fail(c, PTYCHO_ESTATE, "no frame has been appended yet");
        if (alg == PTYCHO_DM && c->present < c->J) return fail(c, PTYCHO_ESTATE, "DM needs every frame (PAPER.md:58); append the rest first");
        CU(cudaStreamWaitEvent(c->stream, c->ev_append, 0));   // the frames appended so far have been copied and re-tiled
    }
    if (alg != PTYCHO_DM) { ptycho_status st = build_batches(c, c->present); if (st != PTYCHO_OK) return st; }
    c->epie_pi = -1;                                        // the probe may have changed since the last call (set_probe, DM, orthogonalisation)
    k_snap_sum_I<<<1, 1, 0, c->stream>>>(c->sc);
    ++c->launches;
    for (int it = 0; it < n_iters; ++it) {
        ptycho_status st = alg == PTYCHO_DM ? dm_iteration(c) : minibatch_iteration(c, alg);
        if (st != PTYCHO_OK) return st;
        double* slot = c->err_hist + (c->t < kErrCap ? c->t : kErrCap - 1);
        LAUNCH(c, PTYCHO_K_UPDATE, (k_sum_error<<<kErrBlocks, 1024, 0, c->stream>>>(c->e_part, (size_t)c->J * ncb_of(c->N), c->sc, slot, c->err_part, c->err_ticket)));
        ++c->t;
    }
    CU(cudaGetLastError());
    return PTYCHO_OK;
}

ptycho_status ptycho_shard_buffers(ptycho_ctx* c, ptycho_shard_bufs* out) {
    if (!c || !out) return PTYCHO_EINVAL;
    if (c->par.shard_total_pos <= 0) return fail(c, PTYCHO_ESTATE, "not a shard (params.shard_total_pos)");
    out->c_canvas = reinterpret_cast<float*>(c->nO);
    out->probe_sums = reinterpret_cast<float*>(c->nP);     // n_P (N^2 complex64) and d_P (N^2 floats) are adjacent for K = 1 (layout)
    if (reinterpret_cast<char*>(c->dP) != reinterpret_cast<char*>(c->nP) + (size_t)c->N * c->N * 8) return fail(c, PTYCHO_ESTATE, "probe sums not adjacent");
    out->sum_I = &c->sc->sum_I;
    out->err_hist = c->err_hist;
    out->row0 = c->shard_row0; out->row1 = c->shard_row1;
    return PTYCHO_OK;
}
ptycho_status ptycho_shard_begin(ptycho_ctx* c) {
    if (!c) return PTYCHO_EINVAL;
    if (c->par.shard_total_pos <= 0) return fail(c, PTYCHO_ESTATE, "not a shard (params.shard_total_pos)");
    if (c->shard_open) return fail(c, PTYCHO_ESTATE, "ptycho_shard_end has not been called");
    k_snap_sum_I<<<1, 1, 0, c->stream>>>(c->sc);
    ++c->launches;
    ptycho_status st = dm_iteration(c, 1);
    if (st != PTYCHO_OK) return st;
    c->shard_open = true;
    return PTYCHO_OK;
}
ptycho_status ptycho_shard_end(ptycho_ctx* c) {
    if (!c) return PTYCHO_EINVAL;
    if (!c->shard_open) return fail(c, PTYCHO_ESTATE, "ptycho_shard_begin has not been called");
    ptycho_status st = dm_iteration(c, 2);
    if (st != PTYCHO_OK) return st;
    double* slot = c->err_hist + (c->t < kErrCap ? c->t : kErrCap - 1);
    LAUNCH(c, PTYCHO_K_UPDATE, (k_sum_error<<<kErrBlocks, 1024, 0, c->stream>>>(c->e_part, (size_t)c->J * ncb_of(c->N), c->sc, slot, c->err_part, c->err_ticket)));
    ++c->t;
    c->shard_open = false;
    CU(cudaGetLastError());
    return PTYCHO_OK;
}

ptycho_status ptycho_fetch_object(ptycho_ctx* c, float* out) {
    if (!c || !out) return PTYCHO_EINVAL;
    CU(cudaMemcpyAsync(out, c->O, (size_t)c->H * c->W * 8, cudaMemcpyDefault, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return PTYCHO_OK;
}
ptycho_status ptycho_fetch_probe(ptycho_ctx* c, float* out) {
    if (!c || !out) return PTYCHO_EINVAL;
    CU(cudaMemcpyAsync(out, c->P, (size_t)c->K * c->N * c->N * 8, cudaMemcpyDefault, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return PTYCHO_OK;
}
ptycho_status ptycho_fetch_error(ptycho_ctx* c, double* out, int cap, int* n_written) {
    if (!c || (!out && cap > 0) || cap < 0) return PTYCHO_EINVAL;
    const int n = std::min(std::min(c->t, cap), kErrCap);
    if (n > 0) CU(cudaMemcpyAsync(out, c->err_hist, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    if (n_written) *n_written = c->t;
    return PTYCHO_OK;
}
ptycho_status ptycho_fetch_steps(ptycho_ctx* c, double* out, int cap, int* n_written) {
    if (!c || (!out && cap > 0) || cap < 0) return PTYCHO_EINVAL;
    const int n = (int)std::min<long long>(std::min<long long>(c->n_steps, cap), kStepCap);
    if (n > 0) CU(cudaMemcpyAsync(out, c->steps, sizeof(double) * 2 * n, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    if (n_written) *n_written = (int)c->n_steps;
    return PTYCHO_OK;
}

ptycho_status ptycho_set_object(ptycho_ctx* c, const float* object) {
    if (!c || !object) return PTYCHO_EINVAL;
    CU(cudaMemcpyAsync(c->O, object, (size_t)c->H * c->W * 8, cudaMemcpyDefault, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return PTYCHO_OK;
}
ptycho_status ptycho_set_probe(ptycho_ctx* c, const float* probe) {
    if (!c || !probe) return PTYCHO_EINVAL;
    CU(cudaMemcpyAsync(c->P, probe, (size_t)c->K * c->N * c->N * 8, cudaMemcpyDefault, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return PTYCHO_OK;
}

// Exit waves move through the scratch S in chunks so that host buffers of any size work.
ptycho_status ptycho_fetch_exit_waves(ptycho_ctx* c, const int32_t* idx, int count, float* out) {
    if (!c || !idx || !out || count < 0) return PTYCHO_EINVAL;
    if (!c->psi || !c->psi_valid) return fail(c, PTYCHO_ESTATE, "no exit waves stored (run DM or set them first)");
    const size_t knn = (size_t)c->K * c->N * c->N;
    std::vector<int> slots(count);
    for (int i = 0; i < count; ++i) {
        if (idx[i] < 0 || idx[i] >= c->J) return fail(c, PTYCHO_EINVAL, "frame index out of range");
        slots[i] = c->slot_of_h[idx[i]];
    }
    for (int s0 = 0; s0 < count; s0 += c->chunk) {
        const int nf = std::min(c->chunk, count - s0);
        CU(cudaMemcpyAsync(c->tmp_idx, slots.data() + s0, nf * 4, cudaMemcpyHostToDevice, c->stream));
        LAUNCH(c, PTYCHO_K_OTHER, (k_copy_frames<<<dim3(64, nf), 256, 0, c->stream>>>(c->S, c->psi, nullptr, c->tmp_idx, knn)));
        CU(cudaMemcpyAsync(out + (size_t)s0 * knn * 2, c->S, (size_t)nf * knn * 8, cudaMemcpyDefault, c->stream));
        CU(cudaStreamSynchronize(c->stream));
    }
    return PTYCHO_OK;
}
ptycho_status ptycho_set_exit_waves(ptycho_ctx* c, const float* psi) {
    if (!c || !psi) return PTYCHO_EINVAL;
    if (!c->psi) return fail(c, PTYCHO_ESTATE, "no exit-wave store (disable_dm was set)");
    const size_t knn = (size_t)c->K * c->N * c->N;
    for (int j0 = 0; j0 < c->J; j0 += c->chunk) {
        const int nf = std::min(c->chunk, c->J - j0);
        CU(cudaMemcpyAsync(c->S, psi + (size_t)j0 * knn * 2, (size_t)nf * knn * 8, cudaMemcpyDefault, c->stream));
        LAUNCH(c, PTYCHO_K_OTHER, (k_copy_frames<<<dim3(64, nf), 256, 0, c->stream>>>(c->psi, c->S, c->slot_of + j0, nullptr, knn)));
    }
    CU(cudaStreamSynchronize(c->stream));
    c->psi_valid = true;
    return PTYCHO_OK;
}

ptycho_status ptycho_revised_waves(ptycho_ctx* c, const int32_t* idx, int count, float* out) {
    if (!c || !idx || !out || count < 0) return PTYCHO_EINVAL;
    if (c->sub_frac) return fail(c, PTYCHO_EUNSUPPORTED, "sub-pixel positions: not available");
    for (int i = 0; i < count; ++i)
        if (idx[i] < 0 || idx[i] >= c->J) return fail(c, PTYCHO_EINVAL, "frame index out of range");
    const size_t knn = (size_t)c->K * c->N * c->N;
    for (int s0 = 0; s0 < count; s0 += c->chunk) {
        const int nf = std::min(c->chunk, count - s0);
        CU(cudaMemcpyAsync(c->tmp_idx, idx + s0, nf * 4, cudaMemcpyHostToDevice, c->stream));
        FrameArgs a = base_args(c);
        a.frames = c->tmp_idx;
        a.e_part = c->e_tmp;
        a.out = c->S;   // in place: every CTA reads its rows of S before it writes them
        passes(c, a, nf, RF_EXIT, CM_FULL, RI_REVISED);
        CU(cudaMemcpyAsync(out + (size_t)s0 * knn * 2, c->S, (size_t)nf * knn * 8, cudaMemcpyDefault, c->stream));
        CU(cudaStreamSynchronize(c->stream));
    }
    return PTYCHO_OK;
}

ptycho_status ptycho_eval_error(ptycho_ctx* c, double* out) {
    if (!c || !out) return PTYCHO_EINVAL;
    if (c->present < c->J) return fail(c, PTYCHO_ESTATE, "eval_error needs every frame");
    if (c->streaming) CU(cudaStreamWaitEvent(c->stream, c->ev_append, 0));
    k_snap_sum_I<<<1, 1, 0, c->stream>>>(c->sc);
    const int ncb = ncb_of(c->N);
    if (c->sub_frac) {                                      // sub-pixel positions (R28): F[P] once, then every launch with its shifted probes
        const size_t knn = (size_t)c->K * c->N * c->N;
        CU(cudaMemcpyAsync(c->sub_FP, c->P, knn * 8, cudaMemcpyDeviceToDevice, c->stream));
        plain_fft2(c, c->sub_FP, c->K, false);
    }
    for (int s0 = 0; s0 < c->J; s0 += c->chunk) {
        const int nf = std::min(c->chunk, c->J - s0);
        FrameArgs a = base_args(c);
        a.frames = c->dm_frames + s0;
        a.e_part = c->e_tmp + (size_t)s0 * ncb;
        if (c->sub_frac) {
            const size_t knn = (size_t)c->K * c->N * c->N;
            LAUNCH(c, PTYCHO_K_OTHER, (k_sub_ramp<<<dim3(nf, (unsigned)((knn + 255) / 256)), 256, 0, c->stream>>>(
                                           c->sub_Pj, c->sub_FP, c->sub_frac, c->dm_frames + s0, c->K, c->N, 1.0f / ((float)c->N * (float)c->N))));
            plain_fft2(c, c->sub_Pj, nf * c->K, true);
            a.Pj = c->sub_Pj;
            passes(c, a, nf, RF_EXIT_PJ, CM_ERRONLY, -1);
        } else
        passes(c, a, nf, RF_EXIT, CM_ERRONLY, -1);
    }
    LAUNCH(c, PTYCHO_K_OTHER, (k_sum_error<<<kErrBlocks, 1024, 0, c->stream>>>(c->e_tmp, (size_t)c->J * ncb, c->sc, c->scratch_d, c->err_part, c->err_ticket)));
    CU(cudaMemcpyAsync(out, c->scratch_d, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return PTYCHO_OK;
}

ptycho_status ptycho_append_frames(ptycho_ctx* c, int first_frame, int count, const void* intensities) {
    if (!c || !intensities || count < 1) return PTYCHO_EINVAL;
    if (!c->streaming) return fail(c, PTYCHO_ESTATE, "not a streaming context (ptycho_init was given the intensities)");
    if (first_frame != c->present || first_frame + count > c->J) return fail(c, PTYCHO_EINVAL, "frames must be appended in order, without gaps");
    const size_t nn = (size_t)c->N * c->N, bpp = c->itype == PTYCHO_I_U16 ? 2 : 4;
    const bool dev = is_device_ptr(intensities);
    cudaStream_t s = c->copy_stream;
    for (int f0 = 0; f0 < count; f0 += c->stage_frames) {
        const int nf = std::min(c->stage_frames, count - f0);
        const char* src = static_cast<const char*>(intensities) + (size_t)f0 * nn * bpp;
        const void* chunk = src;
        if (!dev) { CU(cudaMemcpyAsync(c->stage, src, (size_t)nf * nn * bpp, cudaMemcpyHostToDevice, s)); chunk = c->stage; }
        const dim3 g(nf, ncb_of(c->N));
        const int first = first_frame + f0;
        dispatch_n(c->N, [&](auto nn_) {
            constexpr int NN = decltype(nn_)::value;
            if (c->itype == PTYCHO_I_U16) k_tile_intensity_chunk<NN, unsigned short><<<g, kThreads, 0, s>>>((unsigned short*)c->It, (const unsigned short*)chunk, c->slot_of, first);
            else k_tile_intensity_chunk<NN, float><<<g, kThreads, 0, s>>>((float*)c->It, (const float*)chunk, c->slot_of, first);
        });
        k_sum_intensity<<<kRedBlocks, 256, 0, s>>>(chunk, c->itype, (size_t)nf * nn, c->scratch_s);
        k_finish_sum_I<<<1, 32, 0, s>>>(c->scratch_s, kRedBlocks, c->sc, 1);
        c->launches += 3;
    }
    CU(cudaEventRecord(c->ev_append, s));
    CU(cudaGetLastError());
    c->present += count;
    return PTYCHO_OK;
}
ptycho_status ptycho_wait_frames(ptycho_ctx* c) {
    if (!c) return PTYCHO_EINVAL;
    if (c->copy_stream) CU(cudaStreamSynchronize(c->copy_stream));
    return PTYCHO_OK;
}
int ptycho_frames_present(const ptycho_ctx* c) { return c ? c->present : 0; }

// Hermitian K x K eigenproblem by cyclic complex Jacobi rotations (host, K <= 8).  On return g is diagonal (eigenvalues on the
// diagonal) and the columns of v are the eigenvectors of the input.
static void jacobi_hermitian(int K, std::vector<std::complex<double>>& g, std::vector<std::complex<double>>& v) {
    using cd = std::complex<double>;
    v.assign((size_t)K * K, cd(0, 0));
    for (int i = 0; i < K; ++i) v[i * K + i] = 1.0;
    for (int sweep = 0; sweep < 64; ++sweep) {
        double off = 0, diag = 0;
        for (int p = 0; p < K; ++p) for (int q = 0; q < K; ++q) (p == q ? diag : off) += std::norm(g[p * K + q]);
        if (off <= 1e-30 * diag) break;
        for (int p = 0; p < K; ++p)
            for (int q = p + 1; q < K; ++q) {
                const cd gpq = g[p * K + q];
                const double apq = std::abs(gpq);
                if (apq == 0) continue;
                const cd ph = gpq / apq;                                  // e^{i phi}
                const double app = g[p * K + p].real(), aqq = g[q * K + q].real();
                const double th = 0.5 * std::atan2(2 * apq, app - aqq);
                const double cs = std::cos(th), sn = std::sin(th);
                // rotation R: column p = (cs, sn conj(ph)) , column q = (-sn ph, cs) in rows (p, q)
                for (int k = 0; k < K; ++k) {                              // G <- G R
                    const cd gp = g[k * K + p], gq = g[k * K + q];
                    g[k * K + p] = cs * gp + sn * std::conj(ph) * gq;
                    g[k * K + q] = -sn * ph * gp + cs * gq;
                }
                for (int k = 0; k < K; ++k) {                              // G <- R^H G
                    const cd gp = g[p * K + k], gq = g[q * K + k];
                    g[p * K + k] = cs * gp + sn * ph * gq;
                    g[q * K + k] = -sn * std::conj(ph) * gp + cs * gq;
                }
                for (int k = 0; k < K; ++k) {                              // V <- V R
                    const cd vp = v[k * K + p], vq = v[k * K + q];
                    v[k * K + p] = cs * vp + sn * std::conj(ph) * vq;
                    v[k * K + q] = -sn * ph * vp + cs * vq;
                }
            }
    }
}

ptycho_status ptycho_orthogonalize_modes(ptycho_ctx* c) {
    if (!c) return PTYCHO_EINVAL;
    const int K = c->K, nn = c->N * c->N;
    if (K == 1) return PTYCHO_OK;
    using cd = std::complex<double>;
    double2* part = reinterpret_cast<double2*>(c->scratch_d);             // K*K*kGramBlocks double2 = at most 4096 of its 4736 doubles
    LAUNCH(c, PTYCHO_K_OTHER, (k_gram<<<dim3(K * K, kGramBlocks), 256, 0, c->stream>>>(c->P, K, nn, part)));
    std::vector<double2> hp((size_t)K * K * kGramBlocks);
    CU(cudaMemcpyAsync(hp.data(), part, hp.size() * sizeof(double2), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    std::vector<cd> g((size_t)K * K), v;
    for (int e = 0; e < K * K; ++e) { cd s(0, 0); for (int b = 0; b < kGramBlocks; ++b) s += cd(hp[e * kGramBlocks + b].x, hp[e * kGramBlocks + b].y); g[e] = s; }
    jacobi_hermitian(K, g, v);
    std::vector<int> order(K);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return g[a * K + a].real() > g[b * K + b].real(); });
    MixMatrix U{};
    for (int m = 0; m < K; ++m) {
        const int col = order[m];
        int big = 0;
        for (int i = 1; i < K; ++i) if (std::abs(v[i * K + col]) > std::abs(v[big * K + col])) big = i;
        const cd ph = std::conj(v[big * K + col]) / std::abs(v[big * K + col]);   // makes the largest component real positive
        for (int k = 0; k < K; ++k) { const cd u = std::conj(v[k * K + col] * ph); U.u[m][k] = make_float2((float)u.real(), (float)u.imag()); }   // U = V^H
    }
    LAUNCH(c, PTYCHO_K_OTHER, (k_mix_modes<<<dim3((nn + 255) / 256, 1), 256, 0, c->stream>>>(c->P, K, nn, U)));
    if (c->psi && c->psi_valid)
        LAUNCH(c, PTYCHO_K_OTHER, (k_mix_modes<<<dim3((nn + 255) / 256, c->J), 256, 0, c->stream>>>(c->psi, K, nn, U)));
    CU(cudaStreamSynchronize(c->stream));
    CU(cudaGetLastError());
    return PTYCHO_OK;
}

ptycho_status ptycho_profile(ptycho_ctx* c, int enable) {
    if (!c) return PTYCHO_EINVAL;
    CU(cudaStreamSynchronize(c->stream));
    for (auto& e : c->prof_ev) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
    c->prof_ev.clear();
    for (int i = 0; i < PTYCHO_KCLASS_COUNT; ++i) { c->prof_ms[i] = 0; c->prof_n[i] = 0; }
    c->prof = enable != 0;
    return PTYCHO_OK;
}
ptycho_status ptycho_profile_fetch(ptycho_ctx* c, int kclass, double* total_ms, long long* n_launches) {
    if (!c || kclass < 0 || kclass >= PTYCHO_KCLASS_COUNT) return PTYCHO_EINVAL;
    CU(cudaStreamSynchronize(c->stream));
    for (auto& e : c->prof_ev) {                       // fold finished events into the totals
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, e.a, e.b) == cudaSuccess) { c->prof_ms[e.cls] += ms; ++c->prof_n[e.cls]; }
        cudaEventDestroy(e.a); cudaEventDestroy(e.b);
    }
    c->prof_ev.clear();
    if (total_ms) *total_ms = c->prof_ms[kclass];
    if (n_launches) *n_launches = c->prof_n[kclass];
    return PTYCHO_OK;
}

#ifdef PTYCHO_PHASE_PROF
// debug builds only: copies and clears the phase-cycle counters of dm_mega.cuh
int ptycho_debug_phase(unsigned long long* out16) {
    cudaDeviceSynchronize();
    cudaMemcpyFromSymbol(out16, ptycho::g_phase, 16 * sizeof(unsigned long long));
    unsigned long long z[16] = {};
    cudaMemcpyToSymbol(ptycho::g_phase, z, sizeof(z));
    return 0;
}
#endif

long long ptycho_launch_count(const ptycho_ctx* c) { return c ? c->launches : 0; }
const char* ptycho_last_error(const ptycho_ctx* c) { return c ? c->err.c_str() : g_init_error.c_str(); }
void ptycho_destroy(ptycho_ctx* c) { delete c; }

ptycho_status ptycho_prepare_frames(const void* raw, ptycho_itype raw_type, int n_frames, int det_h, int det_w, int center_y,
                                    int center_x, int n, float threshold, float saturation, int rot90, const float* frame_scale,
                                    void* out, ptycho_itype out_type, void* cuda_stream) {
    ptycho_ctx* c = nullptr;
    if (!raw || !out || n_frames < 1 || det_h < 1 || det_w < 1 || n < 2 || (n & 1)) return PTYCHO_EINVAL;
    if ((raw_type != PTYCHO_I_F32 && raw_type != PTYCHO_I_U16) || (out_type != PTYCHO_I_F32 && out_type != PTYCHO_I_U16)) return PTYCHO_EINVAL;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const size_t in_bytes = (size_t)n_frames * det_h * det_w * (raw_type == PTYCHO_I_U16 ? 2 : 4);
    const size_t total = (size_t)n_frames * n * n, out_bytes = total * (out_type == PTYCHO_I_U16 ? 2 : 4);
    const bool dev_in = is_device_ptr(raw), dev_out = is_device_ptr(out);
    void *d_in = const_cast<void*>(raw), *d_out = out;
    if (rot90 < 0 || rot90 > 3) return PTYCHO_EINVAL;
    struct Tmp { void* p = nullptr; ~Tmp() { if (p) cudaFree(p); } } t_in, t_out, t_sc;   // staging: freed on every return path
    const float* d_sc = frame_scale;
    if (frame_scale && !is_device_ptr(frame_scale)) {
        CU(cudaMalloc(&t_sc.p, (size_t)n_frames * 4));
        CU(cudaMemcpyAsync(t_sc.p, frame_scale, (size_t)n_frames * 4, cudaMemcpyHostToDevice, s));
        d_sc = static_cast<const float*>(t_sc.p);
    }
    if (!dev_in) { CU(cudaMalloc(&t_in.p, in_bytes)); d_in = t_in.p; CU(cudaMemcpyAsync(d_in, raw, in_bytes, cudaMemcpyHostToDevice, s)); }
    if (!dev_out) { CU(cudaMalloc(&t_out.p, out_bytes)); d_out = t_out.p; }
    const bool vec = (n % 16 == 0) && ((reinterpret_cast<uintptr_t>(d_out) & 15) == 0);   // n/2 a multiple of 8: a group of 8 never straddles kx = n/2
    const int grid = (int)std::min<size_t>((total / (vec ? 8 : 1) + 255) / 256, (size_t)148 * 64);
#define PREP(TI, TO) do { if (vec) k_prepare_frames<TI, TO, 8><<<grid, 256, 0, s>>>((const TI*)d_in, det_h, det_w, center_y, center_x, n, threshold, saturation, rot90, d_sc, (TO*)d_out, total); \
                          else k_prepare_frames<TI, TO, 1><<<grid, 256, 0, s>>>((const TI*)d_in, det_h, det_w, center_y, center_x, n, threshold, saturation, rot90, d_sc, (TO*)d_out, total); } while (0)
    if (raw_type == PTYCHO_I_U16 && out_type == PTYCHO_I_U16) PREP(unsigned short, unsigned short);
    else if (raw_type == PTYCHO_I_U16) PREP(unsigned short, float);
    else if (out_type == PTYCHO_I_U16) PREP(float, unsigned short);
    else PREP(float, float);
#undef PREP
    if (!dev_out) CU(cudaMemcpyAsync(out, d_out, out_bytes, cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    CU(cudaGetLastError());
    return PTYCHO_OK;
}

__global__ void k_scale(float2* d, size_t n, float s) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) { d[i].x *= s; d[i].y *= s; }
}

ptycho_status ptycho_test_fft2(float* data, int n, int count, int inverse, void* cuda_stream) {
    if (!data || !valid_n(n) || count < 1) return PTYCHO_EINVAL;
    ptycho_ctx tmp;
    ptycho_ctx* c = &tmp;
    c->N = n; c->K = 1; c->stream = static_cast<cudaStream_t>(cuda_stream);
    ptycho_status st = PTYCHO_OK;
    dispatch_n(n, [&](auto nn) { st = set_attrs<decltype(nn)::value>(c); });
    if (st != PTYCHO_OK) return st;
    std::vector<float2> tw, twi;
    const int E = n == 64 ? 8 : n == 512 ? 32 : 16;
    host_twiddles(n, E, n / E, tw, twi);
    struct Tmp { float2* p = nullptr; ~Tmp() { if (p) cudaFree(p); } } t_tw;   // freed on every return path
    CU(cudaMalloc(&t_tw.p, 2 * n * sizeof(float2)));
    float2* d_tw = t_tw.p;
    CU(cudaMemcpy(d_tw, tw.data(), n * 8, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(d_tw + n, twi.data(), n * 8, cudaMemcpyHostToDevice));
    FrameArgs a{};
    a.S = reinterpret_cast<float2*>(data); a.K = 1; a.tw = d_tw; a.twi = d_tw + n;
    if (!inverse) passes(c, a, count, RF_PLAIN, CM_PLAIN_FWD, -1);
    else {
        passes(c, a, count, -1, CM_PLAIN_INV, RI_PLAIN);
        const size_t tot = (size_t)count * n * n;
        k_scale<<<ew_blocks(tot), 256, 0, c->stream>>>(a.S, tot, 1.0f / ((float)n * n));
    }
    CU(cudaStreamSynchronize(c->stream));
    CU(cudaGetLastError());
    return PTYCHO_OK;
}

}  // extern "C"

// =========================================================================================
// ptycho_fft2_noalloc: the entry point that allocates nothing (include/ptycho_b200.h)
// =========================================================================================
// The scratch of the FFT kernels (forward table, then inverse table) for callers that cannot call cudaMalloc.  In HOST code this
// name is a stand-in, not a device address: the address is taken once per device with cudaGetSymbolAddress (below), with that
// device current, and only that pointer is handed to kernels.
static __device__ __align__(256) float2 g_noalloc_tw[2 * PTYCHO_NOALLOC_MAX_N];

namespace {

constexpr int kNoAllocMaxDevices = 64;
std::mutex g_noalloc_mu;
float2* g_noalloc_ptr[kNoAllocMaxDevices] = {};       // device address of g_noalloc_tw, per device ordinal
unsigned g_noalloc_attrs[kNoAllocMaxDevices] = {};    // per device: bit log2(n) - 6 set once the kernels of size n have their attributes

// The tables of host_twiddles(), written on the device: tw[ka * T + b] = twi[b * E + ka] = exp(-2 pi i b ka / n).
__global__ void k_fill_twiddles(float2* __restrict__ tw, float2* __restrict__ twi, int n, int E, int T) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int ka = i / T, b = i % T;
    const double ang = -2.0 * M_PI * (double)b * ka / n;
    const float2 w = make_float2((float)cos(ang), (float)sin(ang));
    tw[ka * T + b] = w;
    twi[b * E + ka] = w;
}

ptycho_status noalloc_fail(ptycho_status st, const std::string& msg) {
    g_init_error = "ptycho_fft2_noalloc: " + msg;
    return st;
}

}  // namespace

// The static scratch's device address on the current device (taken once per device), the kernels' attributes for size n (once per
// device and size), and this call's twiddle tables written into the scratch on c->stream.
static ptycho_status noalloc_setup(ptycho_ctx* c, int n, float2** tw_out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kNoAllocMaxDevices) return noalloc_fail(PTYCHO_ECUDA, "cudaGetDevice failed or device ordinal >= 64");
    float2* tw = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_noalloc_mu);
        if (!g_noalloc_ptr[dev]) {                         // once per device, with that device current
            void* p = nullptr;
            const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_tw);
            if (e != cudaSuccess || !p) return noalloc_fail(PTYCHO_ECUDA, std::string("cudaGetSymbolAddress: ") + cudaGetErrorString(e));
            g_noalloc_ptr[dev] = static_cast<float2*>(p);
        }
        tw = g_noalloc_ptr[dev];
        const unsigned bit = 1u << (n == 64 ? 0 : n == 128 ? 1 : n == 256 ? 2 : 3);
        if (!(g_noalloc_attrs[dev] & bit)) {               // shared-memory opt-in of the kernels of this size (no allocation)
            ptycho_status st = PTYCHO_OK;
            dispatch_n(n, [&](auto nn) { st = set_attrs<decltype(nn)::value>(c); });
            if (st != PTYCHO_OK) return noalloc_fail(st, c->err);
            g_noalloc_attrs[dev] |= bit;
        }
    }
    const int E = n == 64 ? 8 : n == 512 ? 32 : 16;
    k_fill_twiddles<<<(n + 255) / 256, 256, 0, c->stream>>>(tw, tw + PTYCHO_NOALLOC_MAX_N, n, E, n / E);   // the part of the scratch this call uses
    *tw_out = tw;
    return PTYCHO_OK;
}

extern "C" ptycho_status ptycho_fft2_noalloc(float* data, int n, int count, int inverse, void* cuda_stream) {
    if (n > PTYCHO_NOALLOC_MAX_N)
        return noalloc_fail(PTYCHO_ENOMEM, "n = " + std::to_string(n) + " exceeds the static scratch (PTYCHO_NOALLOC_MAX_N = " + std::to_string(PTYCHO_NOALLOC_MAX_N) + ")");
    if (!data || count < 1) return noalloc_fail(PTYCHO_EINVAL, "null data or count < 1");
    if (!valid_n(n)) return noalloc_fail(PTYCHO_EINVAL, "n must be 64, 128, 256 or 512 (and built into this library)");
    ptycho_ctx tmp;                                        // host-side bookkeeping of the launch helpers only
    ptycho_ctx* c = &tmp;
    c->N = n; c->K = 1; c->stream = static_cast<cudaStream_t>(cuda_stream);
    float2* tw = nullptr;
    {
        const ptycho_status st = noalloc_setup(c, n, &tw);
        if (st != PTYCHO_OK) return st;
    }
    float2* twi = tw + PTYCHO_NOALLOC_MAX_N;
    const size_t nn = (size_t)n * n;
    for (int f0 = 0; f0 < count; f0 += 32768) {            // frames ride in gridDim.y
        const int nf = std::min(32768, count - f0);
        FrameArgs a{};
        a.S = reinterpret_cast<float2*>(data) + (size_t)f0 * nn; a.K = 1; a.tw = tw; a.twi = twi;
        if (!inverse) passes(c, a, nf, RF_PLAIN, CM_PLAIN_FWD, -1);
        else {
            passes(c, a, nf, -1, CM_PLAIN_INV, RI_PLAIN);
            k_scale<<<ew_blocks((size_t)nf * nn), 256, 0, c->stream>>>(a.S, (size_t)nf * nn, 1.0f / ((float)n * n));
        }
    }
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return noalloc_fail(PTYCHO_ECUDA, cudaGetErrorString(e));
    return PTYCHO_OK;
}

// Micro-benchmark entry point (include/ptycho_b200.h): the 1-D FFT of every row, by the product's packed-fp32 line FFT or on the
// tensor cores (fft_mma.cuh).  Allocates nothing (the static scratch above), asynchronous.
extern "C" ptycho_status ptycho_test_fft_rows(float* data, int n, int count, int impl, void* cuda_stream) {
    if (!data || count < 1 || (impl != 0 && impl != 1)) return noalloc_fail(PTYCHO_EINVAL, "ptycho_test_fft_rows: bad argument");
    if (!valid_n(n) || (impl == 1 && n != 256)) return noalloc_fail(PTYCHO_EUNSUPPORTED, "ptycho_test_fft_rows: n must be 64..512 (impl 0) or 256 (impl 1)");
    ptycho_ctx tmp;
    ptycho_ctx* c = &tmp;
    c->N = n; c->K = 1; c->stream = static_cast<cudaStream_t>(cuda_stream);
    if (impl == 1) {
        int dev = 0, sms = 148;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PTYCHO_ECUDA;
        k_rows_mma256<<<sms * 16, 128, 0, c->stream>>>(reinterpret_cast<float2*>(data), (long long)count * n);
    } else {
        float2* tw = nullptr;
        const ptycho_status st = noalloc_setup(c, n, &tw);
        if (st != PTYCHO_OK) return st;
        for (int f0 = 0; f0 < count; f0 += 32768) {
            FrameArgs a{};
            a.S = reinterpret_cast<float2*>(data) + (size_t)f0 * n * n; a.K = 1; a.tw = tw; a.twi = tw + PTYCHO_NOALLOC_MAX_N;
            passes(c, a, std::min(32768, count - f0), RF_PLAIN, -1, -1);
        }
    }
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return noalloc_fail(PTYCHO_ECUDA, cudaGetErrorString(e));
    return PTYCHO_OK;
}
