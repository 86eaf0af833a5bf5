// fengine.cu -- host side of the C ABI declared in include/fengine.h.
//
// Owns the device tables of one engine, validates arguments, and enqueues the kernels of
// fe_fir.cuh / fe_fft.cuh (tiled path) or fe_generic.cuh (shapes the tiled path does not cover)
// on the caller's stream.  No arithmetic of the method runs on the host: twiddle tables, the
// combined rotation*gain table and every step of the path are computed by CUDA kernels.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/fengine.h"
#include "fe_common.cuh"
#include "fe_fft.cuh"
#include "fe_fft2.cuh"
#include "fe_fir.cuh"
#include "fe_fir2.cuh"
#include "fe_fir3.cuh"
#include "fe_generic.cuh"
#include "fe_pipe.cuh"
#include "fe_plans.cuh"
#include "fe_split.cuh"

using namespace fe;

struct fengine {
    int A = 0, n = 0, N = 0, lgN = 0, T = 0, P = 0;
    bool tiled = false;             // tiled kernels cover this (n, T)
    bool packed_ok = false;         // pol-packed kernels (fe_fir2 / fe_fft2) cover this (n, T, P)
    bool pols_equal = true;         // both pols of every antenna have equal coarse delays (needed by them)
    int32_t c_min = 0, c_max = 0;   // range of the coarse delays (host pipeline: which input rows a chunk needs)
    int host_chunks = 8;            // option "host_chunks": pieces of the H2D / compute / D2H pipeline
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
    std::vector<cudaEvent_t> pipe_ev;
    bool allow_packed = true;       // option "pol_packed"
    int64_t n_coarse = 1, n_fine = 1;
    // device tables
    float *d_weights = nullptr;
    int32_t *d_coarse = nullptr;
    float *d_fine_d = nullptr, *d_fine_phi = nullptr;
    float2 *d_gains = nullptr, *d_rg = nullptr;
    float4 *d_tw[3] = {nullptr, nullptr, nullptr};
    float2 *d_tw1s = nullptr, *d_tw2s = nullptr;     // scalar twiddles of the pol-packed FFT
    float4 *d_rg2 = nullptr;                         // pol-interleaved gain (x rotation) table of the pol-packed FFT
    int rg2_mode = -1;                               // -1 stale, 0 const mode, 1 per-spectrum mode
    float2 *d_tpost = nullptr;
    // scratch
    float *d_scratch = nullptr;
    size_t scratch_floats = 0;
    // pipelined kernel (fe_pipe.cuh): L2-resident ring of rows and its control words
    float *d_ring = nullptr;
    size_t ring_floats = 0;
    unsigned int *d_ctl = nullptr;
    size_t ctl_words = 0;
    bool allow_fused = false;       // option "fused": the pipelined kernel (fe_pipe.cuh), slower than the two-kernel path today
    bool scratch_h16 = false;       // option "scratch_fp16": FP16 FIR output / FFT input, not parity grade
    bool fft_h16_attr[2] = {};
    bool l2_persist = false;        // option "l2_persist": launch the two kernels with a persisting L2 window over the scratch
    cudaAccessPolicyWindow l2_win{};
    bool allow_fft2p = false;       // option "fft_persistent": persistent pol-packed FFT with bulk-copy prefetch (fft2p_kernel); measured slower
    bool fft2p_attr[2] = {};
    int opt_split = -1;             // option "split" (fe_split.cuh): -1 = where it wins (n >= 16384), 0 = never, 1 = wherever it exists
    float2 *d_sp_tw1 = nullptr, *d_sp_tw256 = nullptr;   // its twiddle tables
    float4 *d_rg2s = nullptr;                            // d_rg2 in split order (fe_split.cuh: split_gidx)
    float2 *d_sp_ptw1 = nullptr, *d_sp_ptw2 = nullptr;   // n >= 16384: pass twiddles of the n/16-point plan of the pair kernel
    bool split_attr[3] = {};        // shared-memory attribute set (producer, consumer int8, consumer f32)
    int ring_rows = 64;             // option "ring_rows" (D: rows per track, a power of two >= 16); 64 measured best (0.55 ms at config 2; 32: 0.71)
    int opt_fir_warps = 0;          // option "fir_warps" (FIR warps per CTA, 0 = as many as the block allows)
    int opt_tracks = 0;             // option "tracks" (J, 0 = as many as the FIR warps serve)
    int opt_segments = 0;           // option "segments" (K per antenna, 0 = chosen per call)
    int opt_pipe_ctas = 0;          // option "pipe_ctas" (grid, 0 = one CTA per SM)
    unsigned long long *d_stats = nullptr;   // option "pipe_stats": per-CTA clock counters of the pipelined kernel
    bool pipe_attr[2] = {};        // kernel variants whose shared-memory attribute is set on this handle's device
    bool fft_attr[4] = {};          // same for the FFT kernels of the two-kernel path (one plan per handle)
    bool reserved = false;          // fengine_reserve was called: process never allocates afterwards
    int device = 0;
    int n_sms = 0;
    // streaming (fengine_stream_*): user coarse delays, row offset folded into the device table, window buffers
    std::vector<int32_t> h_coarse;
    int64_t stream_off = 0;         // rows the device table is shifted by (0 = not streaming)
    int64_t rows_override = 0;      // rows per stream of the buffer given to process_impl (0 = S + T - 1)
    uint8_t *d_win[2] = {nullptr, nullptr};
    size_t win_bytes = 0;
    int64_t win_H = 0, win_max_new = 0, win_prev_new = 0, win_delay = 0;
    int win_cur = 0;
    int bits = 10;                  // option "sample_bits": width of the packed input samples (4, 8, 10, 12, 16)
    bool rg_dirty = true;
    // staging for fengine_process_host
    uint8_t *d_stage_in = nullptr;
    int8_t *d_stage_out = nullptr;
    size_t stage_in_bytes = 0, stage_out_bytes = 0;
    int8_t *d_rec = nullptr;        // time-major records of fengine_process_heaps
    size_t rec_bytes = 0;
    cudaStream_t host_stream = nullptr;
    // options
    int64_t chunk_spectra = 0;      // 0 = whole call in one chunk
    int fir_rows = 0;               // option "fir_rows": spectra per FIR tile, 0 = chosen per call (fir_rows_for)
    int64_t last_launches = 0;
    bool profile = false;
    std::vector<cudaEvent_t> ev_pool;       // reused events
    std::vector<cudaEvent_t> ev_used;       // triplets (before FIR, between, after FFT) in call order
    std::string err;
};

namespace {

int fail(fengine *fe, int code, const char *fmt, ...)
{
    if (fe) {
        char buf[512];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof buf, fmt, ap);
        va_end(ap);
        fe->err = buf;
    }
    return code;
}

#define FE_CUDA(fe, call)                                                                       \
    do {                                                                                        \
        cudaError_t e_ = (call);                                                                \
        if (e_ != cudaSuccess)                                                                  \
            return fail(fe, FENGINE_ERR_CUDA, "%s failed: %s", #call, cudaGetErrorString(e_)); \
    } while (0)

bool all_finite(const float *p, size_t count)
{
    for (size_t i = 0; i < count; ++i)
        if (!std::isfinite(p[i])) return false;
    return true;
}

bool tiled_n(int n) { return n >= 1024 && n <= 32768; }
bool packed_n(int n) { return n == 1024 || n == 2048 || n == 4096 || n == 8192; }
bool use_packed(const fengine *fe) { return fe->tiled && fe->packed_ok && fe->pols_equal && fe->allow_packed; }
bool tiled_T(int T) { return T == 2 || T == 4 || T == 8 || T == 16 || T == 32; }

template <class Plan>
int build_tables(fengine *fe)
{
    for (int p = 1; p < Plan::q; ++p) {
        const int R = Plan::radix(p), S = Plan::S(p), M = Plan::M(p - 1);
        FE_CUDA(fe, cudaMalloc(&fe->d_tw[p - 1], sizeof(float4) * (size_t)R * S));
        build_pass_twiddles<<<(R * S + 255) / 256, 256>>>(fe->d_tw[p - 1], R, S, M);
    }
    FE_CUDA(fe, cudaMalloc(&fe->d_tpost, sizeof(float2) * (size_t)Plan::n));
    build_post_twiddles<<<(Plan::n + 255) / 256, 256>>>(fe->d_tpost, Plan::n);
    FE_CUDA(fe, cudaGetLastError());
    return FENGINE_OK;
}

template <class Plan>
int build_tables2(fengine *fe)
{
    FE_CUDA(fe, cudaMalloc(&fe->d_tw1s, sizeof(float2) * (size_t)Plan::R1 * Plan::M1));
    build_scalar_twiddles<<<(Plan::R1 * Plan::M1 + 255) / 256, 256>>>(fe->d_tw1s, Plan::R1, Plan::M1, Plan::n);
    FE_CUDA(fe, cudaMalloc(&fe->d_rg2, sizeof(float4) * (size_t)fe->A * Plan::n));
    FE_CUDA(fe, cudaMalloc(&fe->d_tw2s, sizeof(float2) * (size_t)Plan::R2 * Plan::M2));
    build_scalar_twiddles<<<(Plan::R2 * Plan::M2 + 255) / 256, 256>>>(fe->d_tw2s, Plan::R2, Plan::M2, Plan::M1);
    FE_CUDA(fe, cudaGetLastError());
    return FENGINE_OK;
}

// kernel launch with an optional persisting-L2 access-policy window (option "l2_persist": the scratch of an L2-sized
// chunk is rewritten in place chunk after chunk, and lines that persist are not written back in between)
template <class... KArgs, class... Args>
cudaError_t launch_win(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream,
                       const cudaAccessPolicyWindow *win, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    if (win) {
        at[0].id = cudaLaunchAttributeAccessPolicyWindow;
        at[0].val.accessPolicyWindow = *win;
        cfg.attrs = at;
        cfg.numAttrs = 1;
    }
    return cudaLaunchKernelEx(&cfg, kernel, args...);
}

template <class Plan, bool F32OUT>
int launch_fft2(fengine *fe, const Fft2Params &prm, int64_t chunk_len, cudaStream_t stream)
{
    const size_t smem = fft2_smem_bytes<Plan>();
    bool &attr_set = fe->fft_attr[F32OUT ? 1 : 0];      // per handle (= per device), not per process
    if (!attr_set) {
        FE_CUDA(fe, cudaFuncSetAttribute(fft2_kernel<Plan, F32OUT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set = true;
    }
    dim3 grid((unsigned)chunk_len, (unsigned)fe->A);
    if constexpr (Plan::n == 1024 || Plan::n == 4096) {
        if (fe->scratch_h16) {
            bool &attr16 = fe->fft_h16_attr[F32OUT ? 1 : 0];
            if (!attr16) {
                FE_CUDA(fe, cudaFuncSetAttribute(fft2_kernel<Plan, F32OUT, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                attr16 = true;
            }
            fft2_kernel<Plan, F32OUT, true><<<grid, Plan::tpf, smem, stream>>>(prm);
            return FENGINE_OK;
        }
    }
    if (fe->l2_persist)
        FE_CUDA(fe, launch_win(fft2_kernel<Plan, F32OUT>, grid, dim3(Plan::tpf), smem, stream, &fe->l2_win, prm));
    else
        fft2_kernel<Plan, F32OUT><<<grid, Plan::tpf, smem, stream>>>(prm);
    return FENGINE_OK;
}

template <bool F32OUT>
int launch_fft2_n(fengine *fe, const Fft2Params &prm, int64_t chunk_len, cudaStream_t stream)
{
    switch (fe->n) {
    case 1024: return launch_fft2<Plan2_1024, F32OUT>(fe, prm, chunk_len, stream);
    case 2048: return launch_fft2<Plan2_2048, F32OUT>(fe, prm, chunk_len, stream);
    case 4096: return launch_fft2<Plan2_4096, F32OUT>(fe, prm, chunk_len, stream);
    case 8192: return launch_fft2<Plan2_8192, F32OUT>(fe, prm, chunk_len, stream);
    }
    return fail(fe, FENGINE_ERR_INVALID_ARG, "no pol-packed FFT plan for n=%d", fe->n);
}

// Shapes the pol-packed FFT does not cover (n >= 16384) but a pol-packed FIR does: 32 taps (fe_fir3.cuh) and sample
// widths other than 10 bits with 16 taps (fe_fir2.cuh with another sample width) write the scratch in the one-pol FFT's layout, so the tap and
// bit-depth sweeps of the paper (both at 32768 channels) run tiled kernels end to end.
bool use_packed_fir_onepol_fft(const fengine *fe)
{
    if (!fe->tiled || use_packed(fe) || fe->P != 2 || !fe->pols_equal || !fe->allow_packed) return false;
    return (fe->T == 32 && fe->bits == 10) || (fe->T == 16 && fe->bits != 10);
}
bool use_tiled(const fengine *fe)
{
    if (!fe->tiled) return false;
    if (use_packed_fir_onepol_fft(fe)) return true;
    if (fe->bits != 10) return use_packed(fe) && fe->T == 16;
    return fe->T != 32 || use_packed(fe);
}
bool use_fused(const fengine *fe)
{
    return use_packed(fe) && fe->allow_fused && fe->bits == 10 && (fe->T == 2 || fe->T == 4 || fe->T == 8 || fe->T == 16);
}

bool use_split(const fengine *fe)
{
    if (!fe->tiled || !fe->d_sp_tw1 || fe->P != 2 || !fe->pols_equal || !fe->allow_packed || fe->bits != 10) return false;
    if (!split_supported(fe->n, fe->T) || fe->opt_split == 0) return false;
    return fe->opt_split == 1 || split_is_big(fe->n);
}

// Rows per producer tile of the split path: one CTA per SM, so the tile count is chosen for whole waves over the SMs
// against the T - 1 warm-up rows every tile pays.
int split_rows_for(const fengine *fe, int64_t S)
{
    if (fe->fir_rows > 0) return fe->fir_rows;
    const int64_t cols = (int64_t)(fe->n / kSubM) * fe->A;
    double best = -1.0;
    int best_rows = (int)S;
    for (int tiles = 1; tiles <= 64 && tiles <= S; ++tiles) {
        const int64_t rows = (S + tiles - 1) / tiles;
        const int64_t ctas = cols * ((S + rows - 1) / rows);
        const int64_t waves = (ctas + fe->n_sms - 1) / fe->n_sms;
        const double eff = (double)ctas / (double)(waves * fe->n_sms) * (double)rows / (double)(rows + fe->T - 1);
        if (eff > best) {
            best = eff;
            best_rows = (int)rows;
        }
    }
    return best_rows;
}

// ---- pipelined kernel: work decomposition of a call (fe_pipe.cuh) ----
struct PipePlan {
    int FW, J, K, Sseg, D, GP, grid;
    unsigned int total;
    size_t ring_floats, ctl_words;
};

int gcd_int(int a, int b) { return b ? gcd_int(b, a % b) : a; }

PipePlan pipe_plan(const fengine *fe, int64_t S)
{
    PipePlan pl{};
    const int tpf = pipe_team_threads(fe->n);
    const int fw_max = (kPipeMaxThreads - tpf - 64) / 32;                 // team + loader + flow + FIR warps
    pl.FW = fe->opt_fir_warps > 0 ? std::min(fe->opt_fir_warps, fw_max) : fw_max;
    pl.grid = fe->opt_pipe_ctas > 0 ? std::min(fe->opt_pipe_ctas, fe->n_sms) : fe->n_sms;
    const int wpj = fe->n / 32;
    while (pl.grid * pl.FW < wpj && pl.FW < fw_max) ++pl.FW;          // at least one track must fit
    int J = std::max(1, pl.grid * pl.FW / wpj);
    if (fe->opt_tracks > 0) J = std::min(J, fe->opt_tracks);
    // segments per antenna: A * K a multiple of J so that every track runs the same number of jobs, as long as a
    // segment stays long against its T - 1 warm-up rows
    int K = fe->opt_segments > 0 ? fe->opt_segments : J / gcd_int(fe->A, J);
    const int64_t min_rows = 8 * (int64_t)fe->T;
    while (K > 1 && (S + K - 1) / K < min_rows) --K;
    K = (int)std::max<int64_t>(1, std::min<int64_t>(K, S));
    pl.K = K;
    pl.Sseg = (int)((S + K - 1) / K);
    pl.K = (int)((S + pl.Sseg - 1) / pl.Sseg);                         // drop empty trailing segments
    const int n_jobs = fe->A * pl.K;
    pl.J = std::min(J, n_jobs);
    int D = 16;
    while (D < fe->ring_rows) D *= 2;
    pl.D = D;
    // groups per track: track t runs jobs t, t + J, ...; segment k has ceil(len_k / G) groups
    int gp = 0;
    for (int t = 0; t < pl.J; ++t) {
        int g = 0;
        for (int j = t; j < n_jobs; j += pl.J) {
            const int k = j / fe->A;
            const int64_t len = std::min<int64_t>(pl.Sseg, S - (int64_t)k * pl.Sseg);
            g += (int)((len + kPipeG - 1) / kPipeG);
        }
        gp = std::max(gp, g);
    }
    pl.GP = gp;
    pl.total = (unsigned int)gp * (unsigned int)(pl.J * kPipeG);
    pl.ring_floats = (size_t)pl.J * pl.D * fe->N * 2;
    pl.ctl_words = kPipeCtlHeader + 2 * (size_t)pl.J * gp;
    return pl;
}

// ring and control words of the pipelined kernel for a call of S spectra
int ensure_pipe(fengine *fe, const PipePlan &pl)
{
    if (pl.ring_floats > fe->ring_floats) {
        if (fe->reserved) return fail(fe, FENGINE_ERR_STATE, "call needs a larger ring than fengine_reserve sized");
        if (fe->d_ring) {
            FE_CUDA(fe, cudaDeviceSynchronize());
            cudaFree(fe->d_ring);
            fe->d_ring = nullptr;
            fe->ring_floats = 0;
        }
        if (cudaMalloc(&fe->d_ring, pl.ring_floats * sizeof(float)) != cudaSuccess) {
            cudaGetLastError();
            return fail(fe, FENGINE_ERR_ALLOC, "cannot allocate %zu bytes of ring", pl.ring_floats * sizeof(float));
        }
        fe->ring_floats = pl.ring_floats;
    }
    if (pl.ctl_words > fe->ctl_words) {
        if (fe->reserved) return fail(fe, FENGINE_ERR_STATE, "call needs more control words than fengine_reserve sized");
        if (fe->d_ctl) {
            FE_CUDA(fe, cudaDeviceSynchronize());
            cudaFree(fe->d_ctl);
            fe->d_ctl = nullptr;
            fe->ctl_words = 0;
        }
        if (cudaMalloc(&fe->d_ctl, pl.ctl_words * sizeof(unsigned int)) != cudaSuccess) {
            cudaGetLastError();
            return fail(fe, FENGINE_ERR_ALLOC, "cannot allocate the control words of the pipelined kernel");
        }
        fe->ctl_words = pl.ctl_words;
    }
    return FENGINE_OK;
}

int launch_fir2(fengine *fe, const Fir2Params &prm, int64_t chunk_len, cudaStream_t stream, bool onepol = false)
{
    if (fe->T == 32) {                                      // one column per thread: 32 taps stay in registers
        dim3 grid3((unsigned)(fe->N / kFir3Threads), (unsigned)((chunk_len + prm.rows_per_tile - 1) / prm.rows_per_tile),
                   (unsigned)fe->A);
        if (onepol)
            fir3_kernel<32, true><<<grid3, kFir3Threads, 0, stream>>>(prm);
        else
            fir3_kernel<32><<<grid3, kFir3Threads, 0, stream>>>(prm);
        return FENGINE_OK;
    }
    dim3 grid((unsigned)(fe->n / kFir2Threads), (unsigned)((chunk_len + prm.rows_per_tile - 1) / prm.rows_per_tile),
              (unsigned)fe->A);
    if (fe->bits != 10) {                                   // bit-depth sweep: 16 taps only
        if (onepol) {
            switch (fe->bits) {
            case 4: fir2_kernel<16, kFir2OutOnePol, 4><<<grid, kFir2Threads, 0, stream>>>(prm); break;
            case 8: fir2_kernel<16, kFir2OutOnePol, 8><<<grid, kFir2Threads, 0, stream>>>(prm); break;
            case 12: fir2_kernel<16, kFir2OutOnePol, 12><<<grid, kFir2Threads, 0, stream>>>(prm); break;
            case 16: fir2_kernel<16, kFir2OutOnePol, 16><<<grid, kFir2Threads, 0, stream>>>(prm); break;
            default: return fail(fe, FENGINE_ERR_INVALID_ARG, "no tiled FIR for %d-bit samples", fe->bits);
            }
            return FENGINE_OK;
        }
        switch (fe->bits) {
        case 4: fir2_kernel<16, kFir2OutPacked, 4><<<grid, kFir2Threads, 0, stream>>>(prm); break;
        case 8: fir2_kernel<16, kFir2OutPacked, 8><<<grid, kFir2Threads, 0, stream>>>(prm); break;
        case 12: fir2_kernel<16, kFir2OutPacked, 12><<<grid, kFir2Threads, 0, stream>>>(prm); break;
        case 16: fir2_kernel<16, kFir2OutPacked, 16><<<grid, kFir2Threads, 0, stream>>>(prm); break;
        default: return fail(fe, FENGINE_ERR_INVALID_ARG, "no tiled FIR for %d-bit samples", fe->bits);
        }
        return FENGINE_OK;
    }
    if (onepol) return fail(fe, FENGINE_ERR_STATE, "no one-pol-layout variant of the 10-bit pol-packed FIR");
    switch (fe->T) {
    case 2: fir2_kernel<2><<<grid, kFir2Threads, 0, stream>>>(prm); break;
    case 4: fir2_kernel<4><<<grid, kFir2Threads, 0, stream>>>(prm); break;
    case 8: fir2_kernel<8><<<grid, kFir2Threads, 0, stream>>>(prm); break;
    case 16:
        if (fe->scratch_h16)
            fir2_kernel<16, kFir2OutPackedH16><<<grid, kFir2Threads, 0, stream>>>(prm);
        else if (fe->l2_persist)
            FE_CUDA(fe, launch_win(fir2_kernel<16>, grid, dim3(kFir2Threads), 0, stream, &fe->l2_win, prm));
        else
            fir2_kernel<16><<<grid, kFir2Threads, 0, stream>>>(prm);
        break;
    default: return fail(fe, FENGINE_ERR_INVALID_ARG, "no tiled FIR for T=%d", fe->T);
    }
    return FENGINE_OK;
}

template <class Plan, bool F32OUT>
int launch_fft(fengine *fe, const FftParams &prm, int64_t chunk_len, cudaStream_t stream)
{
    const size_t smem = fft_smem_bytes<Plan>(fe->P);
    const size_t smem_max = fft_smem_bytes<Plan>(2);
    bool &attr_set = fe->fft_attr[F32OUT ? 3 : 2];
    if (!attr_set) {
        FE_CUDA(fe, cudaFuncSetAttribute(fft_kernel<Plan, F32OUT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max));
        FE_CUDA(fe, cudaFuncSetAttribute(fft_kernel<Plan, F32OUT>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                         (int)cudaSharedmemCarveoutMaxShared));
        attr_set = true;
    }
    dim3 grid((unsigned)chunk_len, (unsigned)fe->A);
    fft_kernel<Plan, F32OUT><<<grid, Plan::tpf, smem, stream>>>(prm);
    return FENGINE_OK;
}

template <bool F32OUT>
int launch_fft_n(fengine *fe, const FftParams &prm, int64_t chunk_len, cudaStream_t stream)
{
    switch (fe->n) {
    case 1024: return launch_fft<Plan1024, F32OUT>(fe, prm, chunk_len, stream);
    case 2048: return launch_fft<Plan2048, F32OUT>(fe, prm, chunk_len, stream);
    case 4096: return launch_fft<Plan4096, F32OUT>(fe, prm, chunk_len, stream);
    case 8192: return launch_fft<Plan8192, F32OUT>(fe, prm, chunk_len, stream);
    case 16384: return launch_fft<Plan16384, F32OUT>(fe, prm, chunk_len, stream);
    case 32768: return launch_fft<Plan32768, F32OUT>(fe, prm, chunk_len, stream);
    }
    return fail(fe, FENGINE_ERR_INVALID_ARG, "no tiled FFT plan for n=%d", fe->n);
}

int launch_fir(fengine *fe, const FirParams &prm, int64_t chunk_len, cudaStream_t stream)
{
    dim3 grid((unsigned)(fe->N / kFirColsPerBlock), (unsigned)((chunk_len + prm.rows_per_tile - 1) / prm.rows_per_tile),
              (unsigned)(fe->A * fe->P));
    switch (fe->T) {
    case 2: fir_kernel<2><<<grid, kFirThreads, 0, stream>>>(prm); break;
    case 4: fir_kernel<4><<<grid, kFirThreads, 0, stream>>>(prm); break;
    case 8: fir_kernel<8><<<grid, kFirThreads, 0, stream>>>(prm); break;
    case 16: fir_kernel<16><<<grid, kFirThreads, 0, stream>>>(prm); break;
    default: return fail(fe, FENGINE_ERR_INVALID_ARG, "no tiled FIR for T=%d", fe->T);
    }
    return FENGINE_OK;
}

int ensure_scratch(fengine *fe, size_t floats)
{
    if (floats <= fe->scratch_floats) return FENGINE_OK;
    if (fe->reserved) return fail(fe, FENGINE_ERR_STATE, "call needs %zu bytes of scratch, more than fengine_reserve sized", floats * sizeof(float));
    if (fe->d_scratch) {
        FE_CUDA(fe, cudaDeviceSynchronize());
        cudaFree(fe->d_scratch);
        fe->d_scratch = nullptr;
        fe->scratch_floats = 0;
    }
    if (cudaMalloc(&fe->d_scratch, floats * sizeof(float)) != cudaSuccess) {
        cudaGetLastError();
        return fail(fe, FENGINE_ERR_ALLOC, "cannot allocate %zu bytes of scratch", floats * sizeof(float));
    }
    fe->scratch_floats = floats;
    return FENGINE_OK;
}

// Spectra per FIR tile.  A tile of R rows runs R + T steps (T warm-up rows), so long tiles waste less, but the
// grid must still cover the SMs a few times over: 256 rows where the call is large (config 2: 0.147 -> 0.136 ms),
// down to 32 where it is small.
int fir_rows_for(const fengine *fe, int64_t S, int cols_per_cta, int streams_per_cta)
{
    if (fe->fir_rows > 0) return fe->fir_rows;
    const int64_t col_ctas = (int64_t)(fe->N / cols_per_cta) * (fe->A * fe->P / streams_per_cta);
    const int64_t want_ctas = (int64_t)fe->n_sms * 6;
    const int64_t rows = S * col_ctas / want_ctas;
    return (int)std::max<int64_t>(32, std::min<int64_t>(256, rows));
}

GenParams gen_params(const fengine *fe, const void *in, int64_t S)
{
    GenParams g{};
    g.in = static_cast<const uint8_t *>(in);
    g.weights = fe->d_weights;
    g.coarse = fe->d_coarse;
    g.fine_d = fe->d_fine_d;
    g.fine_phi = fe->d_fine_phi;
    g.gains = fe->d_gains;
    g.n_coarse = fe->n_coarse;
    g.n_fine = fe->n_fine;
    g.L = (int64_t)fe->N * (fe->rows_override > 0 ? fe->rows_override : S + fe->T - 1);
    g.stream_bytes = g.L / 8 * fe->bits;
    g.bits = fe->bits;
    g.n_spectra = S;
    g.N = fe->N;
    g.T = fe->T;
    g.P = fe->P;
    g.A = fe->A;
    return g;
}

unsigned gen_grid(const fengine *fe, int64_t total) { return (unsigned)std::min<int64_t>((total + 255) / 256, (int64_t)fe->n_sms * 16); }

// What a call over `Sr` spectra needs besides its inputs and outputs: ONE rule, used by process_impl (which sizes the
// buffers on demand) and by fengine_reserve (which sizes them ahead), so that a reserve for S spectra always covers a
// call of S spectra on the path the handle would take now.
struct CallNeed {
    bool fused;             // the pipelined kernel: an L2 ring and counters (ensure_pipe), no full-size scratch
    bool split;             // fe_split.cuh
    int64_t chunk;          // spectra per scratch-resident chunk
    size_t scratch_floats;  // FP32 words of FIR -> FFT scratch (0 when fused)
};
CallNeed call_need(const fengine *fe, int64_t Sr)
{
    CallNeed c{};
    const size_t streams = (size_t)fe->A * fe->P;
    if (!use_tiled(fe)) {                                   // generic kernels: the whole call at once, chunk_spectra ignored
        c.chunk = Sr;
        c.scratch_floats = streams * (size_t)Sr * fe->N;
        return c;
    }
    c.chunk = fe->chunk_spectra > 0 ? std::min<int64_t>(fe->chunk_spectra, Sr) : Sr;
    c.fused = use_fused(fe) && !fe->scratch_h16;
    c.split = !c.fused && use_split(fe) && !fe->scratch_h16;
    // the n >= 16384 split consumer has the chunk's spectra in gridDim.y (limit 65535): longer calls run in chunks
    if (c.split && split_is_big(fe->n)) c.chunk = std::min<int64_t>(c.chunk, 65535);
    c.scratch_floats = c.fused ? 0 : streams * (size_t)c.chunk * fe->N;
    return c;
}

// every entry point runs on the device the handle was created on
int check_device(fengine *fe)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != fe->device)
        return fail(fe, FENGINE_ERR_STATE, "handle belongs to device %d, current device is %d", fe->device, dev);
    return FENGINE_OK;
}

int check_call(fengine *fe, const void *in, const void *out, int64_t S)
{
    if (!fe) return FENGINE_ERR_INVALID_ARG;
    fe->err.clear();
    if (int rc = check_device(fe)) return rc;
    if (S < 0) return fail(fe, FENGINE_ERR_INVALID_ARG, "n_spectra < 0");
    if (S == 0) return FENGINE_OK;
    if (!in || !out) return fail(fe, FENGINE_ERR_INVALID_ARG, "null device pointer");
    if ((reinterpret_cast<uintptr_t>(in) & 15) || (reinterpret_cast<uintptr_t>(out) & 15))
        return fail(fe, FENGINE_ERR_INVALID_ARG, "in/out must be 16-byte aligned");
    if (fe->n_coarse != 1 && fe->n_coarse < S)
        return fail(fe, FENGINE_ERR_STATE, "coarse delay table has %lld entries per stream, need %lld",
                    (long long)fe->n_coarse, (long long)S);
    if (fe->n_fine != 1 && fe->n_fine < S)
        return fail(fe, FENGINE_ERR_STATE, "fine delay table has %lld entries per stream, need %lld",
                    (long long)fe->n_fine, (long long)S);
    return FENGINE_OK;
}

// The rotation x gain tables depend only on what the setters change, so they are rebuilt there, on the legacy stream,
// and the setter returns after the device has finished: fengine_process never launches a table kernel and a call on
// any stream (blocking or not) sees complete tables.
int refresh_tables(fengine *fe)
{
    const int streams = fe->A * fe->P;
    const bool per_spectrum = fe->n_coarse != 1 || fe->n_fine != 1;
    if (!per_spectrum) {
        dim3 grid((unsigned)((fe->n + 255) / 256), (unsigned)streams);
        build_rg_table<<<grid, 256>>>(fe->d_rg, fe->d_gains, fe->d_coarse, fe->d_fine_d, fe->d_fine_phi, fe->n, streams);
    }
    if (fe->d_rg2) {
        const int mode = per_spectrum ? 1 : 0;
        dim3 grid((unsigned)((fe->n + 255) / 256), (unsigned)fe->A);
        build_rg2_table<<<grid, 256>>>(fe->d_rg2, fe->d_gains, fe->d_coarse, fe->d_fine_d, fe->d_fine_phi, fe->n, fe->A, mode);
        fe->rg2_mode = mode;
        if (fe->d_rg2s) permute_rg2_split<<<grid, 256>>>(fe->d_rg2s, fe->d_rg2, fe->n, 16, fe->A);
    }
    FE_CUDA(fe, cudaGetLastError());
    FE_CUDA(fe, cudaDeviceSynchronize());
    fe->rg_dirty = false;
    return FENGINE_OK;
}

// the whole path; exactly one of out / out_f32 is non-null
// spectra [m_lo, m_hi) of a call of S spectra (m_hi < 0: all of them); a sub-range is only available on the tiled
// two-kernel path (fengine_process_host pipelines over it)
int process_impl(fengine *fe, const void *in, int8_t *out, float *out_f32, int64_t S, cudaStream_t stream,
                 int64_t m_lo = 0, int64_t m_hi = -1)
{
    if (m_hi < 0) m_hi = S;
    if (m_lo == 0) fe->last_launches = 0;
    if (S == 0 || m_hi <= m_lo) return FENGINE_OK;
    if (!use_tiled(fe) && (m_lo != 0 || m_hi != S))
        return fail(fe, FENGINE_ERR_STATE, "sub-range processing needs the tiled kernels");
    const int streams = fe->A * fe->P;

    if (!use_tiled(fe)) {
        int rc = ensure_scratch(fe, call_need(fe, S).scratch_floats);
        if (rc) return rc;
        const GenParams gp = gen_params(fe, in, S);
        gen_fir_kernel<<<gen_grid(fe, (int64_t)streams * S * fe->N), 256, 0, stream>>>(gp, fe->d_scratch);
        if (out_f32)
            gen_dft_kernel<true><<<gen_grid(fe, (int64_t)streams * S * fe->n), 256, 0, stream>>>(gp, fe->d_scratch, nullptr, out_f32);
        else
            gen_dft_kernel<false><<<gen_grid(fe, (int64_t)streams * S * fe->n), 256, 0, stream>>>(gp, fe->d_scratch, out, nullptr);
        fe->last_launches = 2;
        FE_CUDA(fe, cudaGetLastError());
        return FENGINE_OK;
    }

    const bool per_spectrum = fe->n_coarse != 1 || fe->n_fine != 1;
    if (fe->rg_dirty) return fail(fe, FENGINE_ERR_STATE, "rotation / gain tables are stale (a setter failed)");

    const CallNeed need = call_need(fe, m_hi - m_lo);
    const int64_t chunk = need.chunk;
    const bool fused = need.fused, split = need.split;
    if (fe->scratch_h16 && !(use_packed(fe) && fe->bits == 10))
        return fail(fe, FENGINE_ERR_STATE, "scratch_fp16 needs the pol-packed path (equal coarse delays in both pols, 10-bit samples)");

    int rc = fused ? FENGINE_OK : ensure_scratch(fe, need.scratch_floats);
    if (rc) return rc;
    if (fe->l2_persist) {
        int max_win = 0;
        cudaDeviceGetAttribute(&max_win, cudaDevAttrMaxAccessPolicyWindowSize, fe->device);
        fe->l2_win.base_ptr = fe->d_scratch;
        fe->l2_win.num_bytes = std::min<size_t>((size_t)streams * chunk * fe->N * sizeof(float), (size_t)max_win);
        fe->l2_win.hitRatio = 1.0f;
        fe->l2_win.hitProp = cudaAccessPropertyPersisting;
        fe->l2_win.missProp = cudaAccessPropertyStreaming;
    }

    FirParams fp{};
    fp.in = static_cast<const uint8_t *>(in);
    fp.weights = fe->d_weights;
    fp.g = fe->d_scratch;
    fp.coarse = fe->d_coarse;
    fp.n_coarse = fe->n_coarse;
    fp.rows_in = fe->rows_override > 0 ? fe->rows_override : S + fe->T - 1;
    fp.stream_bytes = (int64_t)fe->N * fp.rows_in / 8 * fe->bits;
    fp.chunk_cap = chunk;
    fp.lgN = fe->lgN;
    fp.P = fe->P;
    fp.rows_per_tile = fir_rows_for(fe, m_hi - m_lo, kFirColsPerBlock, 1);

    FftParams xp{};
    xp.g = fe->d_scratch;
    xp.out = out;
    xp.out_f32 = out_f32;
    xp.tab.tw[0] = fe->d_tw[0];
    xp.tab.tw[1] = fe->d_tw[1];
    xp.tab.tw[2] = fe->d_tw[2];
    xp.tab.tpost = fe->d_tpost;
    xp.rg = fe->d_rg;
    xp.gains = fe->d_gains;
    xp.coarse = fe->d_coarse;
    xp.fine_d = fe->d_fine_d;
    xp.fine_phi = fe->d_fine_phi;
    xp.n_coarse = fe->n_coarse;
    xp.n_fine = fe->n_fine;
    xp.chunk_cap = chunk;
    xp.n_spectra = S;
    xp.P = fe->P;
    xp.per_spectrum = per_spectrum ? 1 : 0;

    const bool packed = use_packed(fe);
    const bool fir_packed_only = use_packed_fir_onepol_fft(fe);      // pol-packed FIR in front of the one-pol FFT
    Fir2Params fp2{};
    Fft2Params xp2{};
    if (fir_packed_only) {
        fp2.in = fp.in;
        fp2.weights = fp.weights;
        fp2.g = fp.g;
        fp2.coarse = fp.coarse;
        fp2.n_coarse = fp.n_coarse;
        fp2.stream_bytes = fp.stream_bytes;
        fp2.rows_in = fp.rows_in;
        fp2.chunk_cap = chunk;
        fp2.lgN = fe->lgN;
        fp2.rows_per_tile = fir_rows_for(fe, m_hi - m_lo, 2 * kFir2Threads, 2);
    }
    if (packed || split) {
        fp2.in = fp.in;
        fp2.weights = fp.weights;
        fp2.g = fp.g;
        fp2.coarse = fp.coarse;
        fp2.n_coarse = fp.n_coarse;
        fp2.stream_bytes = fp.stream_bytes;
        fp2.rows_in = fp.rows_in;
        fp2.chunk_cap = chunk;
        fp2.lgN = fe->lgN;
        fp2.rows_per_tile = fir_rows_for(fe, m_hi - m_lo, 2 * kFir2Threads, 2);
        xp2.g = fe->d_scratch;
        xp2.out = out;
        xp2.out_f32 = out_f32;
        xp2.tw1 = fe->d_tw1s;
        xp2.tw2 = fe->d_tw2s;
        xp2.tpost = fe->d_tpost;
        xp2.rg2 = fe->d_rg2;
        xp2.coarse = fe->d_coarse;
        xp2.fine_d = fe->d_fine_d;
        xp2.fine_phi = fe->d_fine_phi;
        xp2.n_coarse = fe->n_coarse;
        xp2.n_fine = fe->n_fine;
        xp2.chunk_cap = chunk;
        xp2.n_spectra = S;
        xp2.per_spectrum = per_spectrum ? 1 : 0;
    }

    if (fused) {
        const int64_t Sr = m_hi - m_lo;
        const PipePlan pl = pipe_plan(fe, Sr);
        rc = ensure_pipe(fe, pl);
        if (rc) return rc;
        PipeParams up{};
        up.fir = fp2;
        up.fft = xp2;
        up.fir.m_begin = up.fft.m_begin = m_lo;
        up.fir.m_end = up.fft.m_end = m_hi;
        up.ring = fe->d_ring;
        up.ctl = fe->d_ctl;
        up.m_lo = m_lo;
        up.S = Sr;
        up.A = fe->A;
        up.K = pl.K;
        up.Sseg = pl.Sseg;
        up.J = pl.J;
        up.wpj = fe->n / 32;
        up.D = pl.D;
        up.GP = pl.GP;
        up.fir_warps = pl.FW;
        up.total_tickets = pl.total;
        up.stats = fe->d_stats;
        cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
        if (fe->profile) {
            for (auto &e : ev) {
                if (fe->ev_pool.empty()) {
                    FE_CUDA(fe, cudaEventCreate(&e));
                } else {
                    e = fe->ev_pool.back();
                    fe->ev_pool.pop_back();
                }
                fe->ev_used.push_back(e);
            }
            FE_CUDA(fe, cudaEventRecord(ev[0], stream));
            FE_CUDA(fe, cudaEventRecord(ev[1], stream));    // no separate FIR launch: the whole step is one kernel
        }
        FE_CUDA(fe, cudaMemsetAsync(fe->d_ctl, 0, sizeof(unsigned int) * pl.ctl_words, stream));
        bool &attr_set = fe->pipe_attr[out_f32 ? 1 : 0];    // (n, T) are fixed per handle; reset when "fir_warps" changes
        cudaError_t ce = pipe_launch(fe->T, fe->n, out_f32 != nullptr, up, pl.grid, !attr_set, stream);
        attr_set = true;
        if (ce != cudaSuccess) return fail(fe, FENGINE_ERR_CUDA, "pipelined kernel launch failed: %s", cudaGetErrorString(ce));
        if (fe->profile) FE_CUDA(fe, cudaEventRecord(ev[2], stream));
        fe->last_launches += 1;
        return FENGINE_OK;
    }

    for (int64_t m0 = m_lo; m0 < m_hi; m0 += chunk) {
        const int64_t m1 = std::min(m_hi, m0 + chunk);
        fp.m_begin = xp.m_begin = fp2.m_begin = xp2.m_begin = m0;
        fp.m_end = xp.m_end = fp2.m_end = xp2.m_end = m1;
        cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
        if (fe->profile) {
            for (auto &e : ev) {
                if (fe->ev_pool.empty()) {
                    FE_CUDA(fe, cudaEventCreate(&e));
                } else {
                    e = fe->ev_pool.back();
                    fe->ev_pool.pop_back();
                }
                fe->ev_used.push_back(e);
            }
            FE_CUDA(fe, cudaEventRecord(ev[0], stream));
        }
        if (split) {
            SplitParams sp{};
            sp.fir = fp2;
            sp.fft = xp2;
            sp.fft.rg2 = fe->d_rg2s;
            sp.fir.rows_per_tile = split_rows_for(fe, m1 - m0);
            sp.tw1 = fe->d_sp_tw1;
            sp.tw256 = fe->d_sp_tw256;
            sp.ptw1 = fe->d_sp_ptw1;
            sp.ptw2 = fe->d_sp_ptw2;
            const dim3 gridp((unsigned)(fe->n / kSubM), (unsigned)((m1 - m0 + sp.fir.rows_per_tile - 1) / sp.fir.rows_per_tile), (unsigned)fe->A);
            cudaError_t ce = split_launch_fir(fe->T, fe->n, sp, gridp, !fe->split_attr[0], stream);
            fe->split_attr[0] = true;
            if (ce != cudaSuccess) return fail(fe, FENGINE_ERR_CUDA, "split producer launch failed: %s", cudaGetErrorString(ce));
            if (fe->profile) FE_CUDA(fe, cudaEventRecord(ev[1], stream));
            bool &attr = fe->split_attr[out_f32 ? 2 : 1];
            const dim3 gridc = split_is_big(fe->n) ? dim3(8u, (unsigned)(m1 - m0), (unsigned)fe->A) : dim3((unsigned)(m1 - m0), (unsigned)fe->A);
            ce = split_launch_fft(fe->n, out_f32 != nullptr, sp, gridc, !attr, stream);
            attr = true;
            if (ce != cudaSuccess) return fail(fe, FENGINE_ERR_CUDA, "split consumer launch failed: %s", cudaGetErrorString(ce));
            if (fe->profile) FE_CUDA(fe, cudaEventRecord(ev[2], stream));
            fe->last_launches += 2;
            continue;
        }
        rc = packed ? launch_fir2(fe, fp2, m1 - m0, stream)
                    : fir_packed_only ? launch_fir2(fe, fp2, m1 - m0, stream, true) : launch_fir(fe, fp, m1 - m0, stream);
        if (rc) return rc;
        if (fe->profile) FE_CUDA(fe, cudaEventRecord(ev[1], stream));
        if (packed && fe->allow_fft2p && fft2p_supported(fe->n) && !fe->scratch_h16) {
            bool &attr = fe->fft2p_attr[out_f32 ? 1 : 0];
            if ((m1 - m0) * (int64_t)fe->A >= ((int64_t)1 << 31))   // the kernel counts (spectrum, antenna) rows in an int
                return fail(fe, FENGINE_ERR_INVALID_ARG, "fft_persistent: more than 2^31 rows in a chunk; set chunk_spectra");
            const int grid = (int)std::min<int64_t>(fe->n_sms, (m1 - m0) * fe->A);
            cudaError_t ce = fft2p_launch(fe->n, out_f32 != nullptr, xp2, fe->A, grid, !attr, stream);
            attr = true;
            if (ce != cudaSuccess) return fail(fe, FENGINE_ERR_CUDA, "persistent FFT launch failed: %s", cudaGetErrorString(ce));
        } else if (packed)
            rc = out_f32 ? launch_fft2_n<true>(fe, xp2, m1 - m0, stream) : launch_fft2_n<false>(fe, xp2, m1 - m0, stream);
        else
            rc = out_f32 ? launch_fft_n<true>(fe, xp, m1 - m0, stream) : launch_fft_n<false>(fe, xp, m1 - m0, stream);
        if (rc) return rc;
        if (fe->profile) FE_CUDA(fe, cudaEventRecord(ev[2], stream));
        fe->last_launches += 2;
    }
    FE_CUDA(fe, cudaGetLastError());
    return FENGINE_OK;
}

}  // namespace

extern "C" {

fengine_t *fengine_create_batched(int n_antennas, int n_channels, int taps, int n_pols, const float *weights)
try {
    if (n_antennas < 1 || n_channels < 8 || n_channels > 32768 || (n_channels & (n_channels - 1)) || taps < 1 ||
        taps > 32 || (n_pols != 1 && n_pols != 2) || !weights)
        return nullptr;
    const int N = 2 * n_channels;
    if (!all_finite(weights, (size_t)N * taps)) return nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return nullptr;                                     // no CPU fallback
    }
    fengine *fe = new (std::nothrow) fengine;
    if (!fe) return nullptr;
    fe->A = n_antennas;
    fe->n = n_channels;
    fe->N = N;
    fe->T = taps;
    fe->P = n_pols;
    while ((1 << fe->lgN) < N) ++fe->lgN;
    fe->tiled = tiled_n(fe->n) && tiled_T(fe->T);
    const size_t streams = (size_t)fe->A * fe->P;
    {
        int dev = 0;
        cudaGetDevice(&dev);
        fe->device = dev;
        cudaDeviceGetAttribute(&fe->n_sms, cudaDevAttrMultiProcessorCount, dev);
        if (fe->n_sms < 1) fe->n_sms = 148;
    }

    bool ok = cudaMalloc(&fe->d_weights, sizeof(float) * (size_t)N * taps) == cudaSuccess &&
              cudaMalloc(&fe->d_coarse, sizeof(int32_t) * streams) == cudaSuccess &&
              cudaMalloc(&fe->d_fine_d, sizeof(float) * streams) == cudaSuccess &&
              cudaMalloc(&fe->d_fine_phi, sizeof(float) * streams) == cudaSuccess &&
              cudaMalloc(&fe->d_gains, sizeof(float2) * streams * fe->n) == cudaSuccess &&
              cudaMalloc(&fe->d_rg, sizeof(float2) * streams * fe->n) == cudaSuccess;
    if (ok) {
        std::vector<float2> ones(streams * fe->n, make_float2(1.f, 0.f));
        ok = cudaMemcpy(fe->d_weights, weights, sizeof(float) * (size_t)N * taps, cudaMemcpyHostToDevice) == cudaSuccess &&
             cudaMemset(fe->d_coarse, 0, sizeof(int32_t) * streams) == cudaSuccess &&
             cudaMemset(fe->d_fine_d, 0, sizeof(float) * streams) == cudaSuccess &&
             cudaMemset(fe->d_fine_phi, 0, sizeof(float) * streams) == cudaSuccess &&
             cudaMemcpy(fe->d_gains, ones.data(), sizeof(float2) * ones.size(), cudaMemcpyHostToDevice) == cudaSuccess;
    }
    if (ok && fe->tiled) {
        int rc = FENGINE_OK;
        switch (fe->n) {
        case 1024: rc = build_tables<Plan1024>(fe); break;
        case 2048: rc = build_tables<Plan2048>(fe); break;
        case 4096: rc = build_tables<Plan4096>(fe); break;
        case 8192: rc = build_tables<Plan8192>(fe); break;
        case 16384: rc = build_tables<Plan16384>(fe); break;
        case 32768: rc = build_tables<Plan32768>(fe); break;
        }
        fe->packed_ok = rc == FENGINE_OK && fe->P == 2 && packed_n(fe->n);
        if (fe->packed_ok) {
            switch (fe->n) {
            case 1024: rc = build_tables2<Plan2_1024>(fe); break;
            case 2048: rc = build_tables2<Plan2_2048>(fe); break;
            case 4096: rc = build_tables2<Plan2_4096>(fe); break;
            case 8192: rc = build_tables2<Plan2_8192>(fe); break;
            }
        }
        if (rc == FENGINE_OK && fe->P == 2 && split_supported(fe->n, fe->T)) {
            const int K1 = 16, M = fe->n / K1;
            bool okm = cudaMalloc(&fe->d_sp_tw1, sizeof(float2) * (size_t)K1 * M) == cudaSuccess &&
                       cudaMalloc(&fe->d_sp_tw256, sizeof(float2) * 256) == cudaSuccess;
            if (okm && !fe->d_rg2) okm = cudaMalloc(&fe->d_rg2, sizeof(float4) * (size_t)fe->A * fe->n) == cudaSuccess;
            if (okm) okm = cudaMalloc(&fe->d_rg2s, sizeof(float4) * (size_t)fe->A * fe->n) == cudaSuccess;
            if (okm) {
                build_scalar_twiddles<<<(K1 * M + 255) / 256, 256>>>(fe->d_sp_tw1, K1, M, fe->n);
                build_scalar_twiddles<<<1, 256>>>(fe->d_sp_tw256, 16, 16, 256);
            }
            if (okm && split_is_big(fe->n)) {                 // the M-point plan of the pair kernel: Plan2_1024 / Plan2_2048
                const int M1 = M / 16, R2 = 8, M2 = M1 / R2;
                okm = cudaMalloc(&fe->d_sp_ptw1, sizeof(float2) * 16 * (size_t)M1) == cudaSuccess &&
                      cudaMalloc(&fe->d_sp_ptw2, sizeof(float2) * (size_t)R2 * M2) == cudaSuccess;
                if (okm) {
                    build_scalar_twiddles<<<(16 * M1 + 255) / 256, 256>>>(fe->d_sp_ptw1, 16, M1, M);
                    build_scalar_twiddles<<<(R2 * M2 + 255) / 256, 256>>>(fe->d_sp_ptw2, R2, M2, M1);
                }
            }
            if (!okm)
                rc = FENGINE_ERR_ALLOC;
            else if (cudaGetLastError() != cudaSuccess)
                rc = FENGINE_ERR_CUDA;
        }
        ok = rc == FENGINE_OK;
    }
    if (ok) ok = cudaDeviceSynchronize() == cudaSuccess;
    if (ok) ok = refresh_tables(fe) == FENGINE_OK;
    if (!ok) {
        cudaGetLastError();
        fengine_destroy(fe);
        return nullptr;
    }
    return fe;
} catch (const std::bad_alloc &) {
    return nullptr;
} catch (...) {
    return nullptr;
}

fengine_t *fengine_create(int n_channels, int taps, int n_pols, const float *weights)
{
    return fengine_create_batched(1, n_channels, taps, n_pols, weights);
}

void fengine_destroy(fengine_t *fe)
{
    if (!fe) return;
    cudaDeviceSynchronize();
    cudaFree(fe->d_weights);
    cudaFree(fe->d_coarse);
    cudaFree(fe->d_fine_d);
    cudaFree(fe->d_fine_phi);
    cudaFree(fe->d_gains);
    cudaFree(fe->d_rg);
    for (auto &t : fe->d_tw) cudaFree(t);
    cudaFree(fe->d_tpost);
    cudaFree(fe->d_tw1s);
    cudaFree(fe->d_tw2s);
    cudaFree(fe->d_rg2);
    cudaFree(fe->d_sp_tw1);
    cudaFree(fe->d_sp_tw256);
    cudaFree(fe->d_rg2s);
    cudaFree(fe->d_sp_ptw1);
    cudaFree(fe->d_sp_ptw2);
    cudaFree(fe->d_scratch);
    cudaFree(fe->d_ring);
    cudaFree(fe->d_ctl);
    cudaFree(fe->d_stats);
    cudaFree(fe->d_win[0]);
    cudaFree(fe->d_win[1]);
    cudaFree(fe->d_rec);
    cudaFree(fe->d_stage_in);
    cudaFree(fe->d_stage_out);
    if (fe->host_stream) cudaStreamDestroy(fe->host_stream);
    if (fe->s_h2d) cudaStreamDestroy(fe->s_h2d);
    if (fe->s_d2h) cudaStreamDestroy(fe->s_d2h);
    for (auto e : fe->pipe_ev) cudaEventDestroy(e);
    for (auto e : fe->ev_pool) cudaEventDestroy(e);
    for (auto e : fe->ev_used) cudaEventDestroy(e);
    cudaGetLastError();
    delete fe;
}

int fengine_set_coarse_delays(fengine_t *fe, const int32_t *c, int64_t n_per_stream)
try {
    if (!fe) return FENGINE_ERR_INVALID_ARG;
    fe->err.clear();
    if (int rc = check_device(fe)) return rc;          // the handle's tables live on its own device
    if (!c || n_per_stream < 1) return fail(fe, FENGINE_ERR_INVALID_ARG, "bad coarse delay table");
    const size_t count = (size_t)fe->A * fe->P * n_per_stream;
    FE_CUDA(fe, cudaDeviceSynchronize());
    if (n_per_stream != fe->n_coarse) {
        int32_t *nd = nullptr;
        if (cudaMalloc(&nd, sizeof(int32_t) * count) != cudaSuccess) {
            cudaGetLastError();
            return fail(fe, FENGINE_ERR_ALLOC, "coarse delay table allocation failed");
        }
        cudaFree(fe->d_coarse);
        fe->d_coarse = nd;
        fe->n_coarse = n_per_stream;
    }
    fe->h_coarse.assign(c, c + count);
    if (fe->stream_off != 0) {                              // streaming: the row offset of the window lives in the table
        std::vector<int32_t> eff(count);
        for (size_t i = 0; i < count; ++i) eff[i] = (int32_t)((int64_t)c[i] - fe->stream_off * fe->N);
        FE_CUDA(fe, cudaMemcpy(fe->d_coarse, eff.data(), sizeof(int32_t) * count, cudaMemcpyHostToDevice));
    } else {
        FE_CUDA(fe, cudaMemcpy(fe->d_coarse, c, sizeof(int32_t) * count, cudaMemcpyHostToDevice));
    }
    fe->c_min = fe->c_max = c[0];
    for (size_t i = 1; i < count; ++i) {
        fe->c_min = std::min(fe->c_min, c[i]);
        fe->c_max = std::max(fe->c_max, c[i]);
    }
    fe->pols_equal = true;                                  // the pol-packed kernels share one delay per antenna
    if (fe->P == 2)
        for (int a = 0; a < fe->A && fe->pols_equal; ++a)
            fe->pols_equal = memcmp(c + (size_t)(2 * a) * n_per_stream, c + (size_t)(2 * a + 1) * n_per_stream,
                                    sizeof(int32_t) * (size_t)n_per_stream) == 0;
    fe->rg_dirty = true;
    return refresh_tables(fe);
} catch (const std::bad_alloc &) {
    return fail(fe, FENGINE_ERR_ALLOC, "out of host memory");
} catch (...) {
    return fail(fe, FENGINE_ERR_CUDA, "unexpected C++ exception");
}

int fengine_set_fine_delays(fengine_t *fe, const float *delay, const float *phase, int64_t n_per_stream)
try {
    if (!fe) return FENGINE_ERR_INVALID_ARG;
    fe->err.clear();
    if (int rc = check_device(fe)) return rc;          // the handle's tables live on its own device
    if (!delay || !phase || n_per_stream < 1) return fail(fe, FENGINE_ERR_INVALID_ARG, "bad fine delay table");
    const size_t count = (size_t)fe->A * fe->P * n_per_stream;
    if (!all_finite(delay, count) || !all_finite(phase, count))
        return fail(fe, FENGINE_ERR_INVALID_ARG, "non-finite fine delay or phase");
    FE_CUDA(fe, cudaDeviceSynchronize());
    if (n_per_stream != fe->n_fine) {
        float *nd = nullptr, *np = nullptr;
        if (cudaMalloc(&nd, sizeof(float) * count) != cudaSuccess || cudaMalloc(&np, sizeof(float) * count) != cudaSuccess) {
            cudaGetLastError();
            cudaFree(nd);
            return fail(fe, FENGINE_ERR_ALLOC, "fine delay table allocation failed");
        }
        cudaFree(fe->d_fine_d);
        cudaFree(fe->d_fine_phi);
        fe->d_fine_d = nd;
        fe->d_fine_phi = np;
        fe->n_fine = n_per_stream;
    }
    FE_CUDA(fe, cudaMemcpy(fe->d_fine_d, delay, sizeof(float) * count, cudaMemcpyHostToDevice));
    FE_CUDA(fe, cudaMemcpy(fe->d_fine_phi, phase, sizeof(float) * count, cudaMemcpyHostToDevice));
    fe->rg_dirty = true;
    return refresh_tables(fe);
} catch (const std::bad_alloc &) {
    return fail(fe, FENGINE_ERR_ALLOC, "out of host memory");
} catch (...) {
    return fail(fe, FENGINE_ERR_CUDA, "unexpected C++ exception");
}

int fengine_set_gains(fengine_t *fe, const float *gains_re_im)
try {
    if (!fe) return FENGINE_ERR_INVALID_ARG;
    fe->err.clear();
    if (int rc = check_device(fe)) return rc;          // the handle's tables live on its own device
    if (!gains_re_im) return fail(fe, FENGINE_ERR_INVALID_ARG, "null gains");
    const size_t count = (size_t)fe->A * fe->P * fe->n;
    if (!all_finite(gains_re_im, count * 2)) return fail(fe, FENGINE_ERR_INVALID_ARG, "non-finite gain");
    FE_CUDA(fe, cudaDeviceSynchronize());
    FE_CUDA(fe, cudaMemcpy(fe->d_gains, gains_re_im, sizeof(float2) * count, cudaMemcpyHostToDevice));
    fe->rg_dirty = true;
    return refresh_tables(fe);
} catch (const std::bad_alloc &) {
    return fail(fe, FENGINE_ERR_ALLOC, "out of host memory");
} catch (...) {
    return fail(fe, FENGINE_ERR_CUDA, "unexpected C++ exception");
}

int fengine_process(fengine_t *fe, const void *in, void *out, int64_t n_spectra, void *stream)
try {
    int rc = check_call(fe, in, out, n_spectra);
    if (rc) return rc;
    if (fe->stream_off != 0) return fail(fe, FENGINE_ERR_STATE, "a stream is open: use fengine_stream_push or fengine_stream_end");
    return process_impl(fe, in, static_cast<int8_t *>(out), nullptr, n_spectra, static_cast<cudaStream_t>(stream));
} catch (const std::bad_alloc &) {
    return fail(fe, FENGINE_ERR_ALLOC, "out of host memory");
} catch (...) {
    return fail(fe, FENGINE_ERR_CUDA, "unexpected C++ exception");
}

int fengine_reserve(fengine_t *fe, int64_t max_spectra)
try {
    if (!fe) return FENGINE_ERR_INVALID_ARG;
    fe->err.clear();
    if (int rc = check_device(fe)) return rc;          // the handle's tables live on its own device
    if (max_spectra < 1) return fail(fe, FENGINE_ERR_INVALID_ARG, "max_spectra < 1");
    fe->reserved = false;                                   // this call may allocate; later process calls may not
    const CallNeed need = call_need(fe, max_spectra);       // the rule process_impl applies to a call of max_spectra
    int rc = FENGINE_OK;
    if (need.fused) {
        // the ring does not depend on S; the counters grow with it (every smaller call needs no more of either)
        rc = ensure_pipe(fe, pipe_plan(fe, max_spectra));
    } else {
        rc = ensure_scratch(fe, need.scratch_floats);
    }
    if (rc) return rc;
    FE_CUDA(fe, cudaDeviceSynchronize());
    fe->reserved = true;
    return FENGINE_OK;
} catch (const std::bad_alloc &) {
    return fail(fe, FENGINE_ERR_ALLOC, "out of host memory");
} catch (...) {
    return fail(fe, FENGINE_ERR_CUDA, "unexpected C++ exception");
}

int fengine_process_heaps(fengine_t *fe, const void *in, void *heaps_out, int64_t n_spectra, void *stream)
try {
    int rc = check_call(fe, in, heaps_out, n_spectra);
    if (rc || n_spectra == 0) return rc;
    if (fe->stream_off != 0) return fail(fe, FENGINE_ERR_STATE, "a stream is open: use fengine_stream_push or fengine_stream_end");
    if (fe->n < 32) return fail(fe, FENGINE_ERR_INVALID_ARG, "heaps need n >= 32");
    const size_t bytes = (size_t)fe->A * n_spectra * fe->n * fe->P * 2;
    if (bytes > fe->rec_bytes) {
        if (fe->d_rec) {
            FE_CUDA(fe, cudaDeviceSynchronize());
            cudaFree(fe->d_rec);
            fe->d_rec = nullptr;
            fe->rec_bytes = 0;
        }
        if (cudaMalloc(&fe->d_rec, bytes) != cudaSuccess) {
            cudaGetLastError();
            return fail(fe, FENGINE_ERR_ALLOC, "cannot allocate %zu bytes for the time-major records", bytes);
        }
        fe->rec_bytes = bytes;
    }
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    rc = process_impl(fe, in, fe->d_rec, nullptr, n_spectra, s);
    if (rc) return rc;
    const int64_t n_heaps = (n_spectra + 255) / 256;
    dim3 grid((unsigned)(fe->n / 32), 8, (unsigned)(fe->A * n_heaps)), block(32, 8);
    if (fe->P == 2 && fe->n % 64 == 0)
        heaps_transpose64_kernel<<<dim3((unsigned)(fe->n / 64), 4, (unsigned)(fe->A * n_heaps)), 256, 0, s>>>(
            reinterpret_cast<const uint32_t *>(fe->d_rec), static_cast<uint32_t *>(heaps_out), n_spectra, fe->n);
    else if (fe->P == 2)
        heaps_transpose_kernel<uint32_t><<<grid, block, 0, s>>>(reinterpret_cast<const uint32_t *>(fe->d_rec),
                                                                static_cast<uint32_t *>(heaps_out), n_spectra, fe->n);
    else
        heaps_transpose_kernel<uint16_t><<<grid, block, 0, s>>>(reinterpret_cast<const uint16_t *>(fe->d_rec),
                                                                static_cast<uint16_t *>(heaps_out), n_spectra, fe->n);
    ++fe->last_launches;
    FE_CUDA(fe, cudaGetLastError());
    return FENGINE_OK;
} catch (const std::bad_alloc &) {
    return fail(fe, FENGINE_ERR_ALLOC, "out of host memory");
} catch (...) {
    return fail(fe, FENGINE_ERR_CUDA, "unexpected C++ exception");
}

// ---- streaming: consecutive pushes continue one sample stream -------------------------------
namespace {
int64_t ceil_div_rows(int64_t x, int lgN) { return x <= 0 ? 0 : (x + ((int64_t)1 << lgN) - 1) >> lgN; }

int upload_coarse(fengine *fe)
{
    const size_t count = (size_t)fe->A * fe->P * fe->n_coarse;
    std::vector<int32_t> eff(count, 0);
    for (size_t i = 0; i < count; ++i)
        eff[i] = (int32_t)((int64_t)(i < fe->h_coarse.size() ? fe->h_coarse[i] : 0) - fe->stream_off * fe->N);
    FE_CUDA(fe, cudaMemcpy(fe->d_coarse, eff.data(), sizeof(int32_t) * count, cudaMemcpyHostToDevice));
    FE_CUDA(fe, cudaDeviceSynchronize());                   // a pageable copy may return before the DMA has landed
    return FENGINE_OK;
}
}  // namespace

int fengine_stream_begin(fengine_t *fe, int64_t max_new_spectra, int64_t *delay_out)
try {
    if (!fe) return FENGINE_ERR_INVALID_ARG;
    fe->err.clear();
    if (int rc = check_device(fe)) return rc;          // the handle's tables live on its own device
    if (max_new_spectra < 1) return fail(fe, FENGINE_ERR_INVALID_ARG, "max_new_spectra < 1");
    FE_CUDA(fe, cudaDeviceSynchronize());
    const int64_t back = ceil_div_rows(fe->c_max, fe->lgN) + 1;       // rows a positive delay (and a lagging column) reach back
    const int64_t fwd = ceil_div_rows(-(int64_t)fe->c_min, fe->lgN);  // rows a negative delay reaches ahead
    fe->win_delay = fe->T - 1 + fwd;
    fe->win_H = fe->win_delay + back;
    fe->win_max_new = max_new_spectra;
    const size_t row_bytes = (size_t)fe->N / 8 * fe->bits;
    const size_t bytes = (size_t)fe->A * fe->P * (size_t)(fe->win_H + max_new_spectra) * row_bytes;
    if (bytes > fe->win_bytes) {
        for (auto &w : fe->d_win) {
            cudaFree(w);
            w = nullptr;
        }
        fe->win_bytes = 0;
        for (auto &w : fe->d_win)
            if (cudaMalloc(&w, bytes) != cudaSuccess) {
                cudaGetLastError();
                return fail(fe, FENGINE_ERR_ALLOC, "cannot allocate %zu bytes for the stream window", bytes);
            }
        fe->win_bytes = bytes;
    }
    FE_CUDA(fe, cudaMemset(fe->d_win[0], 0, fe->win_bytes));         // samples before the stream started are 0 (R3)
    fe->win_cur = 0;
    fe->win_prev_new = 0;
    fe->stream_off = back;
    int rc = upload_coarse(fe);
    if (rc) return rc;
    if (delay_out) *delay_out = fe->win_delay;
    return FENGINE_OK;
} catch (const std::bad_alloc &) {
    return fail(fe, FENGINE_ERR_ALLOC, "out of host memory");
} catch (...) {
    return fail(fe, FENGINE_ERR_CUDA, "unexpected C++ exception");
}

int fengine_stream_push(fengine_t *fe, const void *in_new, void *out, int64_t n_new, void *stream)
try {
    int rc = check_call(fe, in_new, out, n_new);
    if (rc || n_new == 0) return rc;
    if (fe->stream_off == 0) return fail(fe, FENGINE_ERR_STATE, "no stream is open (fengine_stream_begin)");
    if (n_new > fe->win_max_new) return fail(fe, FENGINE_ERR_INVALID_ARG, "more spectra than fengine_stream_begin allowed");
    if (ceil_div_rows(fe->c_max, fe->lgN) + 1 > fe->stream_off || fe->T - 1 + ceil_div_rows(-(int64_t)fe->c_min, fe->lgN) > fe->win_delay)
        return fail(fe, FENGINE_ERR_STATE, "coarse delays set after fengine_stream_begin need more history than it kept");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const size_t rb = (size_t)fe->N / 8 * fe->bits;
    const int n_streams = fe->A * fe->P;
    const int nxt = fe->win_cur ^ 1;
    const size_t pitch_prev = (size_t)(fe->win_H + fe->win_prev_new) * rb, pitch_new = (size_t)(fe->win_H + n_new) * rb;
    // the last H rows of the previous window, then the new rows (the overlap-tail copy of PAPER.md:85-87)
    FE_CUDA(fe, cudaMemcpy2DAsync(fe->d_win[nxt], pitch_new, fe->d_win[fe->win_cur] + (size_t)fe->win_prev_new * rb, pitch_prev,
                                  (size_t)fe->win_H * rb, n_streams, cudaMemcpyDeviceToDevice, s));
    FE_CUDA(fe, cudaMemcpy2DAsync(fe->d_win[nxt] + (size_t)fe->win_H * rb, pitch_new, in_new, (size_t)n_new * rb,
                                  (size_t)n_new * rb, n_streams, cudaMemcpyDeviceToDevice, s));
    fe->rows_override = fe->win_H + n_new;
    rc = process_impl(fe, fe->d_win[nxt], static_cast<int8_t *>(out), nullptr, n_new, s);
    fe->rows_override = 0;
    fe->win_cur = nxt;
    fe->win_prev_new = n_new;
    return rc;
} catch (const std::bad_alloc &) {
    return fail(fe, FENGINE_ERR_ALLOC, "out of host memory");
} catch (...) {
    return fail(fe, FENGINE_ERR_CUDA, "unexpected C++ exception");
}

int fengine_stream_end(fengine_t *fe)
try {
    if (!fe) return FENGINE_ERR_INVALID_ARG;
    fe->err.clear();
    if (int rc = check_device(fe)) return rc;          // the handle's tables live on its own device
    FE_CUDA(fe, cudaDeviceSynchronize());
    fe->stream_off = 0;
    return upload_coarse(fe);
} catch (const std::bad_alloc &) {
    return fail(fe, FENGINE_ERR_ALLOC, "out of host memory");
} catch (...) {
    return fail(fe, FENGINE_ERR_CUDA, "unexpected C++ exception");
}

int fengine_process_host(fengine_t *fe, const void *in_host, void *out_host, int64_t n_spectra)
try {
    if (!fe) return FENGINE_ERR_INVALID_ARG;
    fe->err.clear();
    if (int rc = check_device(fe)) return rc;          // the handle's tables live on its own device
    if (n_spectra < 0) return fail(fe, FENGINE_ERR_INVALID_ARG, "n_spectra < 0");
    if (n_spectra == 0) return FENGINE_OK;
    if (!in_host || !out_host) return fail(fe, FENGINE_ERR_INVALID_ARG, "null host pointer");
    if (fe->stream_off != 0) return fail(fe, FENGINE_ERR_STATE, "a stream is open: use fengine_stream_push or fengine_stream_end");
    const size_t in_bytes = (size_t)fe->A * fe->P * ((size_t)fe->N * (n_spectra + fe->T - 1) / 8 * fe->bits);
    const size_t out_bytes = (size_t)fe->A * n_spectra * fe->n * fe->P * 2;
    if (!fe->host_stream) FE_CUDA(fe, cudaStreamCreateWithFlags(&fe->host_stream, cudaStreamNonBlocking));
    if (in_bytes > fe->stage_in_bytes) {
        cudaFree(fe->d_stage_in);
        fe->d_stage_in = nullptr;
        fe->stage_in_bytes = 0;
        if (cudaMalloc(&fe->d_stage_in, in_bytes) != cudaSuccess) {
            cudaGetLastError();
            return fail(fe, FENGINE_ERR_ALLOC, "input staging allocation failed");
        }
        fe->stage_in_bytes = in_bytes;
    }
    if (out_bytes > fe->stage_out_bytes) {
        cudaFree(fe->d_stage_out);
        fe->d_stage_out = nullptr;
        fe->stage_out_bytes = 0;
        if (cudaMalloc(&fe->d_stage_out, out_bytes) != cudaSuccess) {
            cudaGetLastError();
            return fail(fe, FENGINE_ERR_ALLOC, "output staging allocation failed");
        }
        fe->stage_out_bytes = out_bytes;
    }
    int rc = check_call(fe, fe->d_stage_in, fe->d_stage_out, n_spectra);
    if (rc) return rc;
    // Pipeline (chunks are copied, processed and copied back concurrently): the call is cut into
    // host_chunks pieces of spectra; the input rows a piece needs go up on one stream, the piece is processed on a
    // second and its output records come down on a third, so that PCIe runs in both directions under the kernels.
    const int K = fe->host_chunks;
    if (use_tiled(fe) && K > 1 && n_spectra >= 4 * (int64_t)K) {
        const int64_t S = n_spectra, rows_in = S + fe->T - 1;
        const size_t row_bytes = (size_t)fe->N / 8 * fe->bits, stream_bytes = row_bytes * rows_in;
        const int n_streams = fe->A * fe->P;
        const size_t out_row = (size_t)fe->n * fe->P * 2, out_pitch = out_row * S;
        if (!fe->s_h2d) FE_CUDA(fe, cudaStreamCreateWithFlags(&fe->s_h2d, cudaStreamNonBlocking));
        if (!fe->s_d2h) FE_CUDA(fe, cudaStreamCreateWithFlags(&fe->s_d2h, cudaStreamNonBlocking));
        while (fe->pipe_ev.size() < (size_t)(2 * K)) {
            cudaEvent_t e;
            FE_CUDA(fe, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            fe->pipe_ev.push_back(e);
        }
        // rows of the window of spectrum m: floor((N m - c) / N) .. floor((N m - c + N T - 1) / N)
        const int64_t back = ((int64_t)fe->c_max + fe->N - 1) >> fe->lgN;               // ceil(c_max / N)
        const int64_t fwd = (-(int64_t)fe->c_min + fe->N - 1) >> fe->lgN;               // ceil(-c_min / N)
        (void)back;                                                                     // rows go up in order from 0
        const int64_t per = (S + K - 1) / K;
        int64_t copied = 0;
        int64_t total_launches = 0;
        const uint8_t *src = static_cast<const uint8_t *>(in_host);
        int8_t *dst = static_cast<int8_t *>(out_host);
        for (int k = 0; k * per < S; ++k) {
            const int64_t m0 = k * per, m1 = std::min(S, m0 + per);
            const int64_t need = std::min<int64_t>(rows_in, std::max<int64_t>(0, m1 + fe->T + fwd));
            if (need > copied) {
                FE_CUDA(fe, cudaMemcpy2DAsync(fe->d_stage_in + copied * row_bytes, stream_bytes, src + copied * row_bytes,
                                              stream_bytes, (size_t)(need - copied) * row_bytes, n_streams,
                                              cudaMemcpyHostToDevice, fe->s_h2d));
                copied = need;
            }
            FE_CUDA(fe, cudaEventRecord(fe->pipe_ev[2 * k], fe->s_h2d));
            FE_CUDA(fe, cudaStreamWaitEvent(fe->host_stream, fe->pipe_ev[2 * k], 0));
            rc = process_impl(fe, fe->d_stage_in, fe->d_stage_out, nullptr, S, fe->host_stream, m0, m1);
            if (rc) return rc;
            total_launches += fe->last_launches;
            fe->last_launches = 0;
            FE_CUDA(fe, cudaEventRecord(fe->pipe_ev[2 * k + 1], fe->host_stream));
            FE_CUDA(fe, cudaStreamWaitEvent(fe->s_d2h, fe->pipe_ev[2 * k + 1], 0));
            FE_CUDA(fe, cudaMemcpy2DAsync(dst + m0 * out_row, out_pitch, fe->d_stage_out + m0 * out_row, out_pitch,
                                          (size_t)(m1 - m0) * out_row, fe->A, cudaMemcpyDeviceToHost, fe->s_d2h));
        }
        fe->last_launches = total_launches;
        FE_CUDA(fe, cudaStreamSynchronize(fe->s_h2d));
        FE_CUDA(fe, cudaStreamSynchronize(fe->s_d2h));
        FE_CUDA(fe, cudaStreamSynchronize(fe->host_stream));
        return FENGINE_OK;
    }
    FE_CUDA(fe, cudaMemcpyAsync(fe->d_stage_in, in_host, in_bytes, cudaMemcpyHostToDevice, fe->host_stream));
    rc = process_impl(fe, fe->d_stage_in, fe->d_stage_out, nullptr, n_spectra, fe->host_stream);
    if (rc) return rc;
    FE_CUDA(fe, cudaMemcpyAsync(out_host, fe->d_stage_out, out_bytes, cudaMemcpyDeviceToHost, fe->host_stream));
    FE_CUDA(fe, cudaStreamSynchronize(fe->host_stream));
    return FENGINE_OK;
} catch (const std::bad_alloc &) {
    return fail(fe, FENGINE_ERR_ALLOC, "out of host memory");
} catch (...) {
    return fail(fe, FENGINE_ERR_CUDA, "unexpected C++ exception");
}

int fengine_process_f32(fengine_t *fe, const void *in, float *spectra_out, int64_t n_spectra, void *stream)
try {
    int rc = check_call(fe, in, spectra_out, n_spectra);
    if (rc) return rc;
    if (fe->stream_off != 0) return fail(fe, FENGINE_ERR_STATE, "a stream is open: use fengine_stream_push or fengine_stream_end");
    return process_impl(fe, in, nullptr, spectra_out, n_spectra, static_cast<cudaStream_t>(stream));
} catch (const std::bad_alloc &) {
    return fail(fe, FENGINE_ERR_ALLOC, "out of host memory");
} catch (...) {
    return fail(fe, FENGINE_ERR_CUDA, "unexpected C++ exception");
}

int fengine_debug_unpack(fengine_t *fe, const void *in, int16_t *samples_out, int64_t n_spectra, void *stream)
try {
    int rc = check_call(fe, in, samples_out, n_spectra);
    if (rc || n_spectra == 0) return rc;
    if (fe->stream_off != 0) return fail(fe, FENGINE_ERR_STATE, "a stream is open: the debug hooks see the shifted delay table");
    const GenParams gp = gen_params(fe, in, n_spectra);
    const int64_t total = (int64_t)fe->A * fe->P * n_spectra * fe->N * fe->T;
    gen_unpack_kernel<<<gen_grid(fe, total), 256, 0, static_cast<cudaStream_t>(stream)>>>(gp, samples_out);
    FE_CUDA(fe, cudaGetLastError());
    return FENGINE_OK;
} catch (const std::bad_alloc &) {
    return fail(fe, FENGINE_ERR_ALLOC, "out of host memory");
} catch (...) {
    return fail(fe, FENGINE_ERR_CUDA, "unexpected C++ exception");
}

int fengine_debug_fir(fengine_t *fe, const void *in, float *g_out, int64_t n_spectra, void *stream)
try {
    int rc = check_call(fe, in, g_out, n_spectra);
    if (rc || n_spectra == 0) return rc;
    if (fe->stream_off != 0) return fail(fe, FENGINE_ERR_STATE, "a stream is open: the debug hooks see the shifted delay table");
    if (fe->scratch_h16) return fail(fe, FENGINE_ERR_STATE, "fengine_debug_fir shows the FP32 FIR output: switch scratch_fp16 off");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int64_t total = (int64_t)fe->A * fe->P * n_spectra * fe->N;
    if (!use_tiled(fe)) {
        gen_fir_kernel<<<gen_grid(fe, total), 256, 0, s>>>(gen_params(fe, in, n_spectra), g_out);
    } else if (use_packed(fe) || use_packed_fir_onepol_fft(fe)) {
        rc = ensure_scratch(fe, (size_t)total);
        if (rc) return rc;
        Fir2Params fp{};
        fp.in = static_cast<const uint8_t *>(in);
        fp.weights = fe->d_weights;
        fp.g = fe->d_scratch;
        fp.coarse = fe->d_coarse;
        fp.n_coarse = fe->n_coarse;
        fp.rows_in = n_spectra + fe->T - 1;
        fp.stream_bytes = (int64_t)fe->N * fp.rows_in / 8 * fe->bits;
        fp.m_begin = 0;
        fp.m_end = n_spectra;
        fp.chunk_cap = n_spectra;
        fp.lgN = fe->lgN;
        fp.rows_per_tile = fir_rows_for(fe, n_spectra, 2 * kFir2Threads, 2);
        rc = launch_fir2(fe, fp, n_spectra, s);
        if (rc) return rc;
        unrotate2_kernel<<<gen_grid(fe, total), 256, 0, s>>>(fe->d_scratch, g_out, fe->d_coarse, fe->n_coarse, n_spectra,
                                                         n_spectra, fe->N, fe->A);
    } else {
        rc = ensure_scratch(fe, (size_t)total);
        if (rc) return rc;
        FirParams fp{};
        fp.in = static_cast<const uint8_t *>(in);
        fp.weights = fe->d_weights;
        fp.g = fe->d_scratch;
        fp.coarse = fe->d_coarse;
        fp.n_coarse = fe->n_coarse;
        fp.rows_in = n_spectra + fe->T - 1;
        fp.stream_bytes = (int64_t)fe->N * fp.rows_in / 8 * fe->bits;
        fp.m_begin = 0;
        fp.m_end = n_spectra;
        fp.chunk_cap = n_spectra;
        fp.lgN = fe->lgN;
        fp.P = fe->P;
        fp.rows_per_tile = fir_rows_for(fe, n_spectra, kFirColsPerBlock, 1);
        rc = launch_fir(fe, fp, n_spectra, s);
        if (rc) return rc;
        unrotate_kernel<<<gen_grid(fe, total), 256, 0, s>>>(fe->d_scratch, g_out, fe->d_coarse, fe->n_coarse, n_spectra,
                                                        n_spectra, fe->N, fe->P, fe->A);
    }
    FE_CUDA(fe, cudaGetLastError());
    return FENGINE_OK;
} catch (const std::bad_alloc &) {
    return fail(fe, FENGINE_ERR_ALLOC, "out of host memory");
} catch (...) {
    return fail(fe, FENGINE_ERR_CUDA, "unexpected C++ exception");
}

const char *fengine_last_error(const fengine_t *fe) { return fe ? fe->err.c_str() : "null handle"; }

int fengine_set_option(fengine_t *fe, const char *key, int64_t value)
try {
    if (!fe || !key) return FENGINE_ERR_INVALID_ARG;
    fe->err.clear();
    if (int rc = check_device(fe)) return rc;          // the handle's tables live on its own device
    if (fe->stream_off != 0 && (!strcmp(key, "sample_bits") || !strcmp(key, "force_generic") || !strcmp(key, "pol_packed") ||
                                !strcmp(key, "fused") || !strcmp(key, "split") || !strcmp(key, "scratch_fp16")))
        return fail(fe, FENGINE_ERR_STATE, "option %s changes the data layout or the path and cannot change while a stream is open", key);
    if (!strcmp(key, "chunk_spectra")) {
        if (value < 0) return fail(fe, FENGINE_ERR_INVALID_ARG, "chunk_spectra < 0");
        fe->chunk_spectra = value;
        return FENGINE_OK;
    }
    if (!strcmp(key, "fir_rows")) {
        if (value < 1 || value > 65536) return fail(fe, FENGINE_ERR_INVALID_ARG, "fir_rows out of range");
        fe->fir_rows = (int)value;
        return FENGINE_OK;
    }
    if (!strcmp(key, "profile")) {
        fe->profile = value != 0;
        return FENGINE_OK;
    }
    if (!strcmp(key, "pol_packed")) {
        fe->allow_packed = value != 0;
        return FENGINE_OK;
    }
    if (!strcmp(key, "host_chunks")) {
        if (value < 1 || value > 1024) return fail(fe, FENGINE_ERR_INVALID_ARG, "host_chunks out of range");
        fe->host_chunks = (int)value;
        return FENGINE_OK;
    }
    if (!strcmp(key, "sample_bits")) {
        if (value != 4 && value != 8 && value != 10 && value != 12 && value != 16)
            return fail(fe, FENGINE_ERR_INVALID_ARG, "sample_bits must be 4, 8, 10, 12 or 16");
        fe->bits = (int)value;
        return FENGINE_OK;
    }
    if (!strcmp(key, "fused")) {
        fe->allow_fused = value != 0;
        return FENGINE_OK;
    }
    if (!strcmp(key, "scratch_fp16")) {
        if (value && !(fe->T == 16 && (fe->n == 1024 || fe->n == 4096) && fe->P == 2))
            return fail(fe, FENGINE_ERR_INVALID_ARG, "scratch_fp16 exists for the pol-packed path with T = 16 and n = 1024 or 4096");
        fe->scratch_h16 = value != 0;
        return FENGINE_OK;
    }
    if (!strcmp(key, "l2_persist")) {                       // value = bytes of L2 set aside for persisting lines (0 = off)
        if (value < 0) return fail(fe, FENGINE_ERR_INVALID_ARG, "l2_persist < 0");
        FE_CUDA(fe, cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, (size_t)value));
        fe->l2_persist = value > 0;
        return FENGINE_OK;
    }
    if (!strcmp(key, "fft_persistent")) {
        fe->allow_fft2p = value != 0;
        return FENGINE_OK;
    }
    if (!strcmp(key, "split")) {
        if (value < -1 || value > 1) return fail(fe, FENGINE_ERR_INVALID_ARG, "split must be -1 (auto), 0 or 1");
        fe->opt_split = (int)value;
        return FENGINE_OK;
    }
    if (!strcmp(key, "ring_rows")) {
        if (value < 16 || value > 4096) return fail(fe, FENGINE_ERR_INVALID_ARG, "ring_rows out of range");
        fe->ring_rows = (int)value;
        return FENGINE_OK;
    }
    if (!strcmp(key, "fir_warps") || !strcmp(key, "tracks") || !strcmp(key, "segments") || !strcmp(key, "pipe_ctas")) {
        if (value < 0 || value > 65536) return fail(fe, FENGINE_ERR_INVALID_ARG, "%s out of range", key);
        (key[0] == 'f' ? fe->opt_fir_warps : key[0] == 't' ? fe->opt_tracks : key[0] == 's' ? fe->opt_segments : fe->opt_pipe_ctas) = (int)value;
        fe->pipe_attr[0] = fe->pipe_attr[1] = false;        // the shared-memory size follows fir_warps
        return FENGINE_OK;
    }
    if (!strcmp(key, "pipe_stats")) {                       // 1: allocate and zero the counters; 0: off
        FE_CUDA(fe, cudaDeviceSynchronize());
        cudaFree(fe->d_stats);
        fe->d_stats = nullptr;
        if (value) {
            const size_t bytes = sizeof(unsigned long long) * kStCount * (size_t)fe->n_sms;
            FE_CUDA(fe, cudaMalloc(&fe->d_stats, bytes));
            FE_CUDA(fe, cudaMemset(fe->d_stats, 0, bytes));
        }
        return FENGINE_OK;
    }
    if (!strcmp(key, "force_generic")) {
        fe->tiled = value ? false : (tiled_n(fe->n) && tiled_T(fe->T));
        return FENGINE_OK;
    }
    return fail(fe, FENGINE_ERR_INVALID_ARG, "unknown option %s", key);
} catch (const std::bad_alloc &) {
    return fail(fe, FENGINE_ERR_ALLOC, "out of host memory");
} catch (...) {
    return fail(fe, FENGINE_ERR_CUDA, "unexpected C++ exception");
}

int fengine_profile_read(fengine_t *fe, double *fir_ms, double *fft_ms, int64_t *n_fir, int64_t *n_fft)
try {
    if (!fe) return FENGINE_ERR_INVALID_ARG;
    fe->err.clear();
    if (int rc = check_device(fe)) return rc;          // the handle's tables live on its own device
    double fir = 0.0, fft = 0.0;
    int64_t count = 0;
    for (size_t i = 0; i + 2 < fe->ev_used.size(); i += 3) {
        FE_CUDA(fe, cudaEventSynchronize(fe->ev_used[i + 2]));
        float a = 0.f, b = 0.f;
        FE_CUDA(fe, cudaEventElapsedTime(&a, fe->ev_used[i], fe->ev_used[i + 1]));
        FE_CUDA(fe, cudaEventElapsedTime(&b, fe->ev_used[i + 1], fe->ev_used[i + 2]));
        fir += a;
        fft += b;
        ++count;
    }
    for (auto e : fe->ev_used) fe->ev_pool.push_back(e);
    fe->ev_used.clear();
    if (fir_ms) *fir_ms = fir;
    if (fft_ms) *fft_ms = fft;
    if (n_fir) *n_fir = count;
    if (n_fft) *n_fft = count;
    return FENGINE_OK;
} catch (const std::bad_alloc &) {
    return fail(fe, FENGINE_ERR_ALLOC, "out of host memory");
} catch (...) {
    return fail(fe, FENGINE_ERR_CUDA, "unexpected C++ exception");
}

int64_t fengine_last_launch_count(const fengine_t *fe) { return fe ? fe->last_launches : 0; }

int fengine_debug_pipe_stats(fengine_t *fe, uint64_t *out, int64_t max_words)
{
    if (!fe || !out) return FENGINE_ERR_INVALID_ARG;
    fe->err.clear();
    if (int rc = check_device(fe)) return rc;          // the handle's tables live on its own device
    if (!fe->d_stats) return fail(fe, FENGINE_ERR_STATE, "option pipe_stats is off");
    const int64_t words = std::min<int64_t>(max_words, (int64_t)kStCount * fe->n_sms);
    FE_CUDA(fe, cudaDeviceSynchronize());
    FE_CUDA(fe, cudaMemcpy(out, fe->d_stats, sizeof(uint64_t) * (size_t)words, cudaMemcpyDeviceToHost));
    FE_CUDA(fe, cudaMemset(fe->d_stats, 0, sizeof(unsigned long long) * kStCount * (size_t)fe->n_sms));
    return FENGINE_OK;
}

int fengine_debug_path(const fengine_t *fe)
{
    if (!fe) return -1;
    if (!use_tiled(fe)) return FENGINE_PATH_GENERIC;
    if (use_fused(fe)) return FENGINE_PATH_FUSED;
    if (use_split(fe)) return FENGINE_PATH_SPLIT;
    if (use_packed(fe)) return FENGINE_PATH_POL_PACKED;
    if (use_packed_fir_onepol_fft(fe)) return FENGINE_PATH_PACKED_FIR_ONE_POL_FFT;
    return FENGINE_PATH_ONE_POL;
}

int fengine_debug_fp32_rate(double *lane_ops_per_second, double *ms_out)
{
    if (!lane_ops_per_second) return FENGINE_ERR_INVALID_ARG;
    int dev = 0, n_sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sms < 1) {
        cudaGetLastError();
        return FENGINE_ERR_CUDA;
    }
    float *out = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = FENGINE_ERR_CUDA;
    const int reps = 8;
    if (cudaMalloc(&out, sizeof(float) * 1024 * (size_t)n_sms) == cudaSuccess && cudaEventCreate(&e0) == cudaSuccess &&
        cudaEventCreate(&e1) == cudaSuccess) {
        fp32_rate_kernel<<<n_sms, 1024>>>(out, 1.0f, 0.5f);           // warm-up
        cudaEventRecord(e0);
        for (int r = 0; r < reps; ++r) fp32_rate_kernel<<<n_sms, 1024>>>(out, 1.0f, 0.5f);
        cudaEventRecord(e1);
        float ms = 0.f;
        if (cudaEventSynchronize(e1) == cudaSuccess && cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess && ms > 0.f) {
            const double lane_ops = (double)reps * n_sms * 1024.0 * kRateIters * 16.0 * 2.0;
            *lane_ops_per_second = lane_ops / (ms * 1e-3);
            if (ms_out) *ms_out = ms / reps;
            rc = FENGINE_OK;
        }
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(out);
    cudaGetLastError();
    return rc;
}

}  // extern "C"
