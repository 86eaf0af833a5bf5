// fe_fir.cuh -- steps 1-3 of the path: unpack + coarse delay + polyphase FIR (Eq. (1)).
//
// Data layout.  The input of one stream is viewed as a 2-D array of rows of N samples
// ("a 2D array with width 2n, in which the i-th column undergoes a FIR filter").
// A thread owns one 5-byte group = 4 consecutive *input* columns v0..v0+3 and walks down the rows
// with a T-row sliding window of converted samples in registers and its 4*T weights in registers
// (the paper's register sliding window), so every sample is loaded, unpacked and
// converted exactly once per tile and every tap is one FMA lane-op.
//
// Coarse delay.  With c = N*cq + cr (0 <= cr < N), the sample that Eq. (1)
// pairs with output column t of spectrum m and tap j is row m + j - cq - [t < cr], input column
// v = (t - cr) mod N.  The kernel therefore works in *input* columns (byte-aligned 5-byte groups,
// which is what the paper says pointer arithmetic cannot give for 10-bit samples) and writes the
// row rotated by cr:  g'[v] = g[(v + cr) mod N].  The rotation is undone for free in the
// frequency domain (circular shift theorem): X[k] = exp(-2 pi i k cr / N) * FFT(g')[k], which the
// FFT epilogue folds into the fine-delay phasor.  Columns that wrap (v + cr >= N) read one row
// earlier ("lag"); the single quad that straddles the wrap keeps the previous row's samples too.
//
// Output: scratch rows g' in fp32, one row of N floats per (antenna, spectrum, pol); each group of
// four columns is stored as (g0, g2, g1, g3) so that the FFT's first pass can load the packed
// pair {Re z[i], Re z[i+1]}, {Im z[i], Im z[i+1]} (z[i] = g[2i] + i g[2i+1]) with one
// 128-bit load and no register shuffling.
#pragma once
#include "fe_common.cuh"

namespace fe {

struct FirParams {
    const uint8_t *in;        // [A*P][stream_bytes]
    const float *weights;     // [N*T], weights[t + N*j] = w[t][j]
    float *g;                 // scratch, row (a*chunk_cap + (m - m_begin))*P + p, N floats
    const int32_t *coarse;    // [A*P][n_coarse]
    int64_t n_coarse;
    int64_t stream_bytes;
    int64_t rows_in;          // S_total + T - 1
    int64_t m_begin, m_end;   // spectra [m_begin, m_end) of this launch
    int64_t chunk_cap;        // scratch rows per antenna per pol
    int lgN;
    int P;
    int rows_per_tile;
};

constexpr int kFirThreads = 128;
constexpr int kFirColsPerThread = 4;
constexpr int kFirColsPerBlock = kFirThreads * kFirColsPerThread;   // 512

// 5 bytes (big-endian bit stream) -> 4 sign-extended samples.  W0/W1 are the two little-endian
// aligned words that contain the group; sel picks bytes b0..b3 as a big-endian word.
__device__ __forceinline__ void unpack_quad(uint32_t W0, uint32_t W1, uint32_t sel, float (&s)[4])
{
    const uint32_t be = __byte_perm(W0, W1, sel);               // b0 b1 b2 b3  = stream bits 39..8
    const uint32_t be2 = __byte_perm(W0, W1, sel + 0x1111u);    // b1 b2 b3 b4  = stream bits 31..0
    s[0] = (float)((int32_t)be >> 22);                          // bits 39..30
    s[1] = (float)((int32_t)(be << 10) >> 22);                  // bits 29..20
    s[2] = (float)((int32_t)(be2 << 12) >> 22);                 // bits 19..10
    s[3] = (float)((int32_t)(be2 << 22) >> 22);                 // bits  9..0
}

template <int T, int PF>
__device__ __forceinline__ void fir_run(const FirParams &prm, const uint8_t *sbase, int64_t c, int64_t m0,
                                        int n_out, int v0, float *grow0)
{
    static_assert(T % PF == 0, "prefetch depth must divide the tap count");
    const int N = 1 << prm.lgN;
    const int cr = (int)(c & (int64_t)(N - 1));
    const int64_t cq = (c - cr) >> prm.lgN;

    // output columns, lag flags and weights of this thread's four input columns
    bool lag[4];
    f2 wA[T], wB[T];                                            // (col0, col2), (col1, col3)
    {
        int tc[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int t = v0 + i + cr;
            lag[i] = t >= N;
            tc[i] = t & (N - 1);
        }
#pragma unroll
        for (int j = 0; j < T; ++j) {
            wA[j] = f2(__ldg(prm.weights + tc[0] + (size_t)N * j), __ldg(prm.weights + tc[2] + (size_t)N * j));
            wB[j] = f2(__ldg(prm.weights + tc[1] + (size_t)N * j), __ldg(prm.weights + tc[3] + (size_t)N * j));
        }
    }
    const bool mixed = lag[3] && !lag[0];
    const int64_t base_row = m0 - cq - (lag[0] ? 1 : 0);        // input row of ring step 0
    // valid ring steps: 0 <= base_row + rho < rows_in
    const int64_t lo64 = -base_row, hi64 = prm.rows_in - base_row;
    const int rho_lo = (int)max((int64_t)-1, min(lo64, (int64_t)0x3fffffff));
    const int rho_hi = (int)max((int64_t)-1, min(hi64, (int64_t)0x3fffffff));

    const int row_words = (N / 4 * 5) / 4;                      // row stride in 32-bit words
    const int64_t byte0 = base_row * (int64_t)(N / 4 * 5) + (int64_t)(v0 / 4) * 5;
    const uint32_t sh = (uint32_t)(byte0 & 3);
    const uint32_t sel = (sh + 3) | ((sh + 2) << 4) | ((sh + 1) << 8) | (sh << 12);
    const uint32_t *wp = reinterpret_cast<const uint32_t *>(sbase) + (byte0 >> 2);   // word of step 0

    auto fetch = [&](int rho, uint32_t &W0, uint32_t &W1) {
        if (rho >= rho_lo && rho < rho_hi) {
            const uint32_t *q = wp + (int64_t)rho * row_words;
            W0 = __ldg(q);
            W1 = __ldg(q + 1);
        } else {
            W0 = 0u;
            W1 = 0u;
        }
    };

    float prev[4] = {0.f, 0.f, 0.f, 0.f};
    if (mixed) {                                                // the quad that straddles the wrap
        uint32_t W0, W1;
        fetch(-1, W0, W1);
        unpack_quad(W0, W1, sel, prev);
    }

    uint32_t raw0[PF], raw1[PF];
#pragma unroll
    for (int k = 0; k < PF; ++k) fetch(k, raw0[k], raw1[k]);

    f2 rA[T], rB[T];                                            // sliding window, slot = rho mod T

    auto insert = [&](int slot_pf, int rho, f2 &dstA, f2 &dstB) {
        float s[4];
        unpack_quad(raw0[slot_pf], raw1[slot_pf], sel, s);
        fetch(rho + PF, raw0[slot_pf], raw1[slot_pf]);          // refill the prefetch slot
        if (mixed) {
            float t[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                t[i] = lag[i] ? prev[i] : s[i];
                prev[i] = s[i];
            }
            dstA = f2(t[0], t[2]);
            dstB = f2(t[1], t[3]);
        } else {
            dstA = f2(s[0], s[2]);
            dstB = f2(s[1], s[3]);
        }
    };

    // warm-up: rows 0 .. T-2
#pragma unroll
    for (int rho = 0; rho < T - 1; ++rho) insert(rho % PF, rho, rA[rho], rB[rho]);

    float4 *gp = reinterpret_cast<float4 *>(grow0 + v0);
    const size_t g_stride4 = ((size_t)N * prm.P) / 4;           // next spectrum, same pol (float4 units)

    for (int i0 = 0; i0 < n_out; i0 += T) {
#pragma unroll
        for (int ii = 0; ii < T; ++ii) {
            if (i0 + ii < n_out) {
                constexpr int dummy = 0;
                (void)dummy;
                const int slot = (ii + T - 1) % T;
                insert(slot % PF, i0 + ii + T - 1, rA[slot], rB[slot]);
                f2 a0 = rA[ii % T] * wA[0], b0 = rB[ii % T] * wB[0];
                f2 a1, b1;
                if (T > 1) {
                    a1 = rA[(ii + 1) % T] * wA[1];
                    b1 = rB[(ii + 1) % T] * wB[1];
                }
#pragma unroll
                for (int j = 2; j < T; j += 2) {
                    a0 = fma_(rA[(ii + j) % T], wA[j], a0);
                    b0 = fma_(rB[(ii + j) % T], wB[j], b0);
                    if (j + 1 < T) {
                        a1 = fma_(rA[(ii + j + 1) % T], wA[j + 1], a1);
                        b1 = fma_(rB[(ii + j + 1) % T], wB[j + 1], b1);
                    }
                }
                if (T > 1) {
                    a0 = a0 + a1;
                    b0 = b0 + b1;
                }
                // (g0, g2, g1, g3)
                stg_stream_f4(gp, make_float4(a0.v.x, a0.v.y, b0.v.x, b0.v.y));
                gp += g_stride4;
            }
        }
    }
}

template <int T, int PF>
__global__ void __launch_bounds__(kFirThreads) fir_kernel(const FirParams prm)
{
    const int N = 1 << prm.lgN;
    const int stream = blockIdx.z;
    const int a = stream / prm.P, p = stream - a * prm.P;
    const int v0 = (blockIdx.x * kFirThreads + threadIdx.x) * kFirColsPerThread;
    int64_t m = prm.m_begin + (int64_t)blockIdx.y * prm.rows_per_tile;
    const int64_t m_stop = min(m + (int64_t)prm.rows_per_tile, prm.m_end);
    const uint8_t *sbase = prm.in + (int64_t)stream * prm.stream_bytes;
    const int32_t *ctab = prm.coarse + (int64_t)stream * prm.n_coarse;

    while (m < m_stop) {
        const int32_t c = ctab[prm.n_coarse == 1 ? 0 : m];
        int64_t run_end = m_stop;
        if (prm.n_coarse != 1) {
            run_end = m + 1;
            while (run_end < m_stop && ctab[run_end] == c) ++run_end;
        }
        float *grow0 = prm.g + (((int64_t)a * prm.chunk_cap + (m - prm.m_begin)) * prm.P + p) * (int64_t)N;
        fir_run<T, PF>(prm, sbase, (int64_t)c, m, (int)(run_end - m), v0, grow0);
        m = run_end;
    }
}

}  // namespace fe
