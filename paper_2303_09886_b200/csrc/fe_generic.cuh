// fe_generic.cuh -- simple one-thread-per-output CUDA kernels.
//
// They serve (a) the debug hooks of include/fengine.h, (b) shapes the tiled kernels do not cover
// (tiny n used by brute-force parity tests, tap counts other than 2/4/8/16, n = 2^k not in the
// plan list).  They are still the CUDA path (no CPU fallback), just not the fast one.
#pragma once
#include "fe_common.cuh"

namespace fe {

// sample u of a packed stream of `bits`-bit two's complement samples (big-endian bit stream, 10 bits in
// the paper's deployment, 4..16 in its bit-depth sweep PAPER.md:273-279), 0 outside [0, L)
__device__ __forceinline__ int gen_sample(const uint8_t *s, int64_t L, int64_t u, int bits)
{
    if (u < 0 || u >= L) return 0;
    const int64_t bit = (int64_t)bits * u, nbytes = (L * bits) >> 3;
    const int64_t B = bit >> 3;
    const int off = (int)(bit & 7);
    uint32_t w = (uint32_t)s[B] << 16;                               // 24-bit window holding the sample
    if (B + 1 < nbytes) w |= (uint32_t)s[B + 1] << 8;
    if (B + 2 < nbytes) w |= (uint32_t)s[B + 2];
    const int v = (int)((w >> (24 - off - bits)) & ((1u << bits) - 1u));
    const int sign = 1 << (bits - 1);
    return (v ^ sign) - sign;
}

struct GenParams {
    const uint8_t *in;
    const float *weights;
    const int32_t *coarse;
    const float *fine_d, *fine_phi;
    const float2 *gains;
    int64_t n_coarse, n_fine;
    int64_t stream_bytes, L, n_spectra;
    int N, T, P, A;
    int bits;                 // sample width of the packed input
};

// debug: window samples [A][P][S][N*T] int16
static __global__ void gen_unpack_kernel(const GenParams p, int16_t *out)
{
    const int64_t NT = (int64_t)p.N * p.T;
    const int64_t total = (int64_t)p.A * p.P * p.n_spectra * NT;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = idx % NT;
        const int64_t m = (idx / NT) % p.n_spectra;
        const int64_t st = idx / NT / p.n_spectra;
        const int64_t c = p.coarse[st * p.n_coarse + (p.n_coarse == 1 ? 0 : m)];
        out[idx] = (int16_t)gen_sample(p.in + st * p.stream_bytes, p.L, (int64_t)p.N * m - c + i, p.bits);
    }
}

// Eq. (1), natural column order: g [A][P][S][N]
static __global__ void gen_fir_kernel(const GenParams p, float *g)
{
    const int64_t total = (int64_t)p.A * p.P * p.n_spectra * p.N;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (int64_t)gridDim.x * blockDim.x) {
        const int t = (int)(idx % p.N);
        const int64_t m = (idx / p.N) % p.n_spectra;
        const int64_t st = idx / p.N / p.n_spectra;
        const int64_t c = p.coarse[st * p.n_coarse + (p.n_coarse == 1 ? 0 : m)];
        const uint8_t *s = p.in + st * p.stream_bytes;
        float acc = 0.f;
        for (int j = 0; j < p.T; ++j) {
            const int64_t u = (int64_t)p.N * (m + j) - c + t;
            acc = fmaf((float)gen_sample(s, p.L, u, p.bits), p.weights[t + (int64_t)p.N * j], acc);
        }
        g[idx] = acc;
    }
}

// N-point DFT of g (natural order, [A][P][S][N]) + rotation + gain (+ quantise): one thread per channel
template <bool F32OUT>
static __global__ void gen_dft_kernel(const GenParams p, const float *g, int8_t *out, float *out_f32)
{
    const int n = p.N / 2;
    const int64_t total = (int64_t)p.A * p.P * p.n_spectra * n;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (int64_t)gridDim.x * blockDim.x) {
        const int k = (int)(idx % n);
        const int64_t m = (idx / n) % p.n_spectra;
        const int64_t st = idx / n / p.n_spectra;
        const int a = (int)(st / p.P), pol = (int)(st % p.P);
        const float *row = g + (st * p.n_spectra + m) * p.N;
        double xr = 0.0, xi = 0.0;
        for (int t = 0; t < p.N; ++t) {
            const int e = (int)(((int64_t)k * t) % p.N);
            double s, c;
            sincospi(-2.0 * (double)e / (double)p.N, &s, &c);
            xr += (double)row[t] * c;
            xi += (double)row[t] * s;
        }
        const double d = (double)p.fine_d[st * p.n_fine + (p.n_fine == 1 ? 0 : m)];
        const double phi = (double)p.fine_phi[st * p.n_fine + (p.n_fine == 1 ? 0 : m)];
        double s1, c1, s2, c2;
        sincospi(-2.0 * d * (double)k / (double)p.N, &s1, &c1);
        sincos(phi, &s2, &c2);
        const double rr = c1 * c2 - s1 * s2, ri = c1 * s2 + s1 * c2;
        const double ur = xr * rr - xi * ri, ui = xr * ri + xi * rr;
        const float2 G = p.gains[st * n + k];
        const float yr = (float)(ur * (double)G.x - ui * (double)G.y);
        const float yi = (float)(ur * (double)G.y + ui * (double)G.x);
        const int64_t o = ((((int64_t)a * p.n_spectra + m) * n + k) * p.P + pol) * 2;
        if (F32OUT) {
            out_f32[o] = yr;
            out_f32[o + 1] = yi;
        } else {
            out[o] = (int8_t)__float2int_rn(fminf(fmaxf(yr, -127.f), 127.f));
            out[o + 1] = (int8_t)__float2int_rn(fminf(fmaxf(yi, -127.f), 127.f));
        }
    }
}

// debug: undo the rotation and the quad permutation of the tiled FIR's scratch rows:
// g_out [A][P][S][N] (natural) from g' rows ((a*cap + m)*P + p)
static __global__ void unrotate_kernel(const float *gp, float *g_out, const int32_t *coarse, int64_t n_coarse,
                                int64_t n_spectra, int64_t cap, int N, int P, int A)
{
    const int64_t total = (int64_t)A * P * n_spectra * N;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (int64_t)gridDim.x * blockDim.x) {
        const int t = (int)(idx % N);
        const int64_t m = (idx / N) % n_spectra;
        const int64_t st = idx / N / n_spectra;
        const int a = (int)(st / P), pol = (int)(st % P);
        const int64_t c = coarse[st * n_coarse + (n_coarse == 1 ? 0 : m)];
        const int cr = (int)(c & (int64_t)(N - 1));
        const int v = (t - cr) & (N - 1);
        const int i = v & 3;
        const int pos = (v & ~3) + (i == 1 ? 2 : i == 2 ? 1 : i);      // stored as (g0, g2, g1, g3)
        g_out[idx] = gp[(((int64_t)a * cap + m) * P + pol) * N + pos];
    }
}

// Channel-major output heaps: the X-engines consume, per antenna and per group of 256 spectra,
// a [channel][256 spectra][pol] array of Gaussian integers.  rec is the time-major output [A][S][n] of words
// (one word = the P (re, im) byte pairs of a channel), heaps is [A][ceil(S/256)][n][256] words; spectra past S in
// the last heap are zero.  32 x 32-word tiles through shared memory, both sides coalesced.
template <typename Word>
static __global__ void heaps_transpose_kernel(const Word *__restrict__ rec, Word *__restrict__ heaps, int64_t S, int n)
{
    __shared__ Word tile[32][33];
    const int64_t n_heaps = (S + 255) / 256;
    const int a = blockIdx.z / (int)n_heaps, h = blockIdx.z - a * (int)n_heaps;
    const int k0 = blockIdx.x * 32, s0 = blockIdx.y * 32;             // channel / in-heap spectrum of the tile
    const Word *src = rec + ((int64_t)a * S + (int64_t)h * 256) * n;
    Word *dst = heaps + ((int64_t)a * n_heaps + h) * (int64_t)n * 256;
    for (int j = threadIdx.y; j < 32; j += blockDim.y) {
        const int64_t m = (int64_t)h * 256 + s0 + j;
        tile[j][threadIdx.x] = m < S ? src[(int64_t)(s0 + j) * n + k0 + threadIdx.x] : Word(0);
    }
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += blockDim.y)
        dst[(int64_t)(k0 + j) * 256 + s0 + threadIdx.x] = tile[threadIdx.x][j];
}


// The same transposition for 4-byte words (two pols) and n a multiple of 64: 64 x 64-word tiles, 256 threads, every
// global access 16 bytes wide (four channels on the way in, four spectra on the way out), 256 contiguous bytes per
// 16 lanes on both sides; the tile rows are 65 words apart so that neither phase has a bank conflict.
static __global__ void __launch_bounds__(256) heaps_transpose64_kernel(const uint32_t *__restrict__ rec, uint32_t *__restrict__ heaps,
                                                                      int64_t S, int n)
{
    __shared__ uint32_t tile[64][65];
    const int64_t n_heaps = (S + 255) / 256;
    const int a = blockIdx.z / (int)n_heaps, h = blockIdx.z - a * (int)n_heaps;
    const int k0 = blockIdx.x * 64, s0 = blockIdx.y * 64;             // channel / in-heap spectrum of the tile
    const uint32_t *src = rec + ((int64_t)a * S + (int64_t)h * 256) * n;
    uint32_t *dst = heaps + ((int64_t)a * n_heaps + h) * (int64_t)n * 256;
    const int q = threadIdx.x & 15, r = threadIdx.x >> 4;
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        const int j = r + 16 * p;                                     // spectrum of the tile
        const int64_t m = (int64_t)h * 256 + s0 + j;
        uint4 v = make_uint4(0u, 0u, 0u, 0u);
        if (m < S) v = *reinterpret_cast<const uint4 *>(src + (int64_t)(s0 + j) * n + k0 + 4 * q);
        tile[j][4 * q] = v.x;
        tile[j][4 * q + 1] = v.y;
        tile[j][4 * q + 2] = v.z;
        tile[j][4 * q + 3] = v.w;
    }
    __syncthreads();
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        const int c = r + 16 * p;                                     // channel of the tile
        const uint4 v = make_uint4(tile[4 * q][c], tile[4 * q + 1][c], tile[4 * q + 2][c], tile[4 * q + 3][c]);
        stg_stream_u4(reinterpret_cast<uint4 *>(dst + (int64_t)(k0 + c) * 256 + s0 + 4 * q), v);
    }
}

// Measurement hook (fengine_debug_fp32_rate): the FIR's instruction form, one sample pair against 16 scalar weights
// into 16 accumulator pairs (FFMA2, the sample operand reused), in a loop that does nothing else.  What it sustains is
// the denominator of the "alu" roofline of bench.py; the path's butterflies (FADD2 / FMUL2)
// issue at the same rate, an FFMA2 with three fresh operands at about three quarters of it.
constexpr int kRateIters = 2048;
static __global__ void __launch_bounds__(1024, 1) fp32_rate_kernel(float *out, float a0, float b0)
{
    float2 acc[16];
    float w[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        acc[i] = make_float2(threadIdx.x * 1e-3f + i, i * 0.5f);
        w[i] = b0 + i * 0.01f + threadIdx.x * 1e-7f;
    }
    float2 s = make_float2(a0 + threadIdx.x * 1e-6f, a0 - 1.0f);
    for (int it = 0; it < kRateIters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) acc[i] = __ffma2_rn(s, make_float2(w[i], w[i]), acc[i]);
        s.x = -s.x;
    }
    float r = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) r += acc[i].x + acc[i].y;
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}

}  // namespace fe
