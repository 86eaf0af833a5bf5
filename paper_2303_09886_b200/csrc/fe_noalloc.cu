// fe_noalloc.cu -- fengine_process_noalloc: the whole path (steps 1-7) for callers that are not
// allowed to allocate device memory.
//
// Who that is.  fengine_create and the first fengine_process of a handle call cudaMalloc (tables, the FIR -> FFT
// scratch).  Some users of this library cannot do that: code that runs after the application has handed all of the
// GPU's memory to its own pool, a real-time receive loop (chunks must be processed as fast as they
// arrive) in which the implicit device-wide synchronisation and the unbounded latency of cudaMalloc / cudaFree are not
// acceptable, or a plug-in whose host forbids allocations after start-up.  For them this file offers one call that
// takes every table as a DEVICE pointer the caller already owns and keeps the only intermediate of the path -- the FIR
// output g of Eq. (1), which the transform reads back -- in an array that is part of the library image.
//
// The scratch array.  `noalloc_scratch` below is a file-scope __device__ array of FENGINE_NOALLOC_MAX_FLOATS floats
// (4 MiB).  It is created when the CUDA module of this library is loaded on a device and every GPU that loads the
// library holds it until the process exits; nothing here calls cudaMalloc, cudaFree or an allocating library routine.
// In HOST code the name `noalloc_scratch` is only a stand-in the runtime uses to look the array up; it is not a device
// address and must never be handed to a kernel.  The device address is asked for once per device, with that device
// current, by cudaGetSymbolAddress (scratch_for_current_device below); the first call on a device does this, so make
// that first call outside any stream capture.
//
// Sharing.  Every call on a device uses the same array and the array keeps what the last call left in it.  Nothing has
// to start at zero: the FIR kernel writes all A*P*S*N words the transform kernel reads, on the same stream, before it
// reads them.  Two calls whose kernels can overlap on the GPU (different streams without an event between them,
// different host threads) race on the array and both results are undefined: order them.
//
// The kernels are the one-thread-per-output kernels of fe_generic.cuh (the path fengine_process takes with option
// "force_generic"), here given the built-in array instead of the handle's cudaMalloc'ed scratch; the output is
// therefore identical to that path's.  They are simple, not fast: this entry point is for small, latency-critical or
// allocation-free use, not for the throughput figures of bench.py.
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/fengine.h"
#include "fe_generic.cuh"

namespace {

// the FIR -> transform intermediate of fengine_process_noalloc; 256-byte aligned so that rows start on full sectors
static __device__ __align__(256) float noalloc_scratch[FENGINE_NOALLOC_MAX_FLOATS];

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
float *g_scratch_ptr[kMaxDevices] = {};     // device address of noalloc_scratch on device i (null = not looked up yet)
int g_n_sms[kMaxDevices] = {};

int report(char *err, int64_t err_len, int code, const char *fmt, ...)
{
    if (err && err_len > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err, (size_t)err_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// One-time set-up per device (the device that is current): the device address of the built-in array and the SM count.
// No allocation: cudaGetSymbolAddress only looks the symbol up in the module the runtime has loaded for this device.
int scratch_for_current_device(float **ptr, int *n_sms, char *err, int64_t err_len)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return report(err, err_len, FENGINE_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices)
        return report(err, err_len, FENGINE_ERR_STATE, "device index %d is outside the %d devices this call supports", dev, kMaxDevices);
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_ptr[dev]) {
        float *p = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void **>(&p), noalloc_scratch);
        if (e != cudaSuccess || !p)
            return report(err, err_len, FENGINE_ERR_CUDA, "cudaGetSymbolAddress(noalloc_scratch) on device %d: %s", dev,
                          cudaGetErrorString(e));
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || sms <= 0)
            return report(err, err_len, FENGINE_ERR_CUDA, "cudaDeviceGetAttribute(SM count) on device %d: %s", dev, cudaGetErrorString(e));
        g_n_sms[dev] = sms;
        g_scratch_ptr[dev] = p;
    }
    *ptr = g_scratch_ptr[dev];
    *n_sms = g_n_sms[dev];
    return FENGINE_OK;
}

}  // namespace

extern "C" int fengine_process_noalloc(const void *in, void *out, const float *weights, const int32_t *coarse_delays,
                                       const float *fine_delays, const float *phases, const float *gains_re_im,
                                       int n_antennas, int n_channels, int taps, int n_pols, int64_t n_spectra,
                                       void *stream, char *err, int64_t err_len)
{
    try {
        if (err && err_len > 0) err[0] = '\0';
        const int n = n_channels, T = taps, P = n_pols, A = n_antennas;
        if (n < 8 || n > 32768 || (n & (n - 1)))
            return report(err, err_len, FENGINE_ERR_INVALID_ARG, "n_channels = %d: need a power of two in [8, 32768]", n);
        if (T < 1 || T > 32) return report(err, err_len, FENGINE_ERR_INVALID_ARG, "taps = %d: need 1 <= taps <= 32", T);
        if (P < 1 || P > 2) return report(err, err_len, FENGINE_ERR_INVALID_ARG, "n_pols = %d: need 1 or 2", P);
        if (A < 1) return report(err, err_len, FENGINE_ERR_INVALID_ARG, "n_antennas = %d: need >= 1", A);
        if (n_spectra < 0) return report(err, err_len, FENGINE_ERR_INVALID_ARG, "n_spectra < 0");
        const int64_t N = 2 * (int64_t)n, S = n_spectra;
        // A*P*S*N <= the array, tested without overflow (A*P*N alone fits easily in 64 bits)
        const int64_t per_spectrum = (int64_t)A * P * N;
        if (per_spectrum > (int64_t)FENGINE_NOALLOC_MAX_FLOATS || S > (int64_t)FENGINE_NOALLOC_MAX_FLOATS / per_spectrum)
            return report(err, err_len, FENGINE_ERR_INVALID_ARG,
                          "the call needs n_antennas * n_pols * n_spectra * 2 * n_channels = %lld x %lld floats of scratch; the "
                          "built-in array holds FENGINE_NOALLOC_MAX_FLOATS = %lld (at most %lld spectra for this shape): split "
                          "the batch, or use fengine_process where allocating is allowed",
                          (long long)per_spectrum, (long long)S, (long long)FENGINE_NOALLOC_MAX_FLOATS,
                          (long long)((int64_t)FENGINE_NOALLOC_MAX_FLOATS / per_spectrum));
        if (S == 0) return FENGINE_OK;
        if (!in || !out || !weights || !coarse_delays || !fine_delays || !phases || !gains_re_im)
            return report(err, err_len, FENGINE_ERR_INVALID_ARG, "null device pointer");
        if ((reinterpret_cast<uintptr_t>(weights) | reinterpret_cast<uintptr_t>(coarse_delays) |
             reinterpret_cast<uintptr_t>(fine_delays) | reinterpret_cast<uintptr_t>(phases)) & 3)
            return report(err, err_len, FENGINE_ERR_INVALID_ARG, "weights / coarse_delays / fine_delays / phases must be 4-byte aligned");
        if (reinterpret_cast<uintptr_t>(gains_re_im) & 7)
            return report(err, err_len, FENGINE_ERR_INVALID_ARG, "gains_re_im must be 8-byte aligned");

        float *scratch = nullptr;
        int n_sms = 0;
        if (int rc = scratch_for_current_device(&scratch, &n_sms, err, err_len)) return rc;

        fe::GenParams gp{};
        gp.in = static_cast<const uint8_t *>(in);
        gp.weights = weights;
        gp.coarse = coarse_delays;
        gp.fine_d = fine_delays;
        gp.fine_phi = phases;
        gp.gains = reinterpret_cast<const float2 *>(gains_re_im);
        gp.n_coarse = 1;
        gp.n_fine = 1;
        gp.L = N * (S + T - 1);
        gp.bits = 10;
        gp.stream_bytes = gp.L / 8 * gp.bits;
        gp.n_spectra = S;
        gp.N = (int)N;
        gp.T = T;
        gp.P = P;
        gp.A = A;

        cudaStream_t s = static_cast<cudaStream_t>(stream);
        const int64_t cap = (int64_t)n_sms * 16;
        const int64_t n_g = per_spectrum * S, n_x = n_g / 2;
        const unsigned grid_g = (unsigned)((n_g + 255) / 256 < cap ? (n_g + 255) / 256 : cap);
        const unsigned grid_x = (unsigned)((n_x + 255) / 256 < cap ? (n_x + 255) / 256 : cap);
        fe::gen_fir_kernel<<<grid_g, 256, 0, s>>>(gp, scratch);                                  // g -> built-in array
        fe::gen_dft_kernel<false><<<grid_x, 256, 0, s>>>(gp, scratch, static_cast<int8_t *>(out), nullptr);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return report(err, err_len, FENGINE_ERR_CUDA, "kernel launch: %s", cudaGetErrorString(e));
        return FENGINE_OK;
    } catch (...) {
        return report(err, err_len, FENGINE_ERR_CUDA, "unexpected exception");
    }
}
