// fe_fir.cuh -- steps 1-3 of the path: unpack + coarse delay + polyphase FIR (Eq. (1)).
//
// Data layout.  The input of one stream is viewed as a 2-D array of rows of N samples
// ("a 2D array with width 2n, in which the i-th column undergoes a FIR filter").
// A thread owns one 5-byte group = 4 consecutive *input* columns v0..v0+3 and walks down the rows
// with a T-row sliding window of converted samples in registers and its 4*T weights in registers
// (the paper's register sliding window), so every sample is loaded, unpacked and
// converted exactly once per tile and every tap is one FMA lane-op (issued as packed FFMA2).
//
// Input staging.  Each warp owns a small ring of rows in shared memory (160 bytes per row: 32
// lanes x 5 bytes) that it fills with 16-byte cp.async copies kDepth-1 rows ahead of use, so the
// HBM/L2 latency is hidden without spending registers, and every global access is an aligned
// 128-bit one (BASELINE.json north_star (a)).
//
// Coarse delay.  With c = N*cq + cr (0 <= cr < N), the sample that Eq. (1)
// pairs with output column t of spectrum m and tap j is row m + j - cq - [t < cr], input column
// v = (t - cr) mod N.  The kernel therefore works in *input* columns (byte-aligned 5-byte groups,
// which is what the paper says pointer arithmetic cannot give for 10-bit samples) and writes the
// row rotated by cr:  g'[v] = g[(v + cr) mod N].  The rotation is undone for free in the
// frequency domain (circular shift theorem): X[k] = exp(-2 pi i k cr / N) * FFT(g')[k], which the
// FFT epilogue folds into the fine-delay phasor.  Columns that wrap (v + cr >= N) read one row
// earlier ("lag"): a thread whose four columns all lag reads the ring one slot behind; the single
// quad that straddles the wrap (MIXED) reads both slots.
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
constexpr int kFirWarps = kFirThreads / 32;
constexpr int kFirColsPerThread = 4;
constexpr int kFirColsPerBlock = kFirThreads * kFirColsPerThread;   // 512
constexpr int kFirRowBytes = 160;                                   // per warp per row: 32 lanes x 5 bytes
constexpr int kFirDepth = 8;                                        // ring slots per warp

__device__ __forceinline__ void cp_async_16(uint32_t smem_addr, const void *gptr)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_addr), "l"(gptr) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N_PENDING>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N_PENDING) : "memory"); }

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

// One run of n_out consecutive spectra with a constant coarse delay c, for this thread's quad.
//   ring      this warp's shared-memory ring, kFirDepth slots of kFirRowBytes
//   wsrc      global address of byte 0 of this warp's 160-byte segment in input row 0 of the stream
//
// Ring step q of the warp holds input row R0 + q, R0 = m0 - cq - 1, and every lane consumes the ring
// steps in order, one per loop step, into its T-row register window.  After ring step q >= T-1 the
// window holds rows R0+q-T+1 .. R0+q, which is spectrum q-T of the run for a column without lag and
// spectrum q-T+1 for a lagging column: lagging columns simply run one spectrum ahead, so the inner
// loop is identical for every lane and only the store row (and its bounds predicate) differs.
template <int T>
__device__ __forceinline__ void fir_run(const FirParams &prm, const uint8_t *wsrc, uint32_t ring_s, int64_t c,
                                        int64_t m0, int n_out, int v0, float *grow0)
{
    constexpr int D = kFirDepth;
    static_assert(D >= 4, "ring too shallow");
    const int N = 1 << prm.lgN;
    const int lane = threadIdx.x & 31;
    const int cr = (int)(c & (int64_t)(N - 1));
    const int64_t cq = (c - cr) >> prm.lgN;

    // output columns, lag flags and weights of this thread's four input columns
    int lagi[4];
    f2 wA[T], wB[T];                                            // (col0, col2), (col1, col3)
    {
        int tc[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int t = v0 + i + cr;
            lagi[i] = t >= N ? 1 : 0;
            tc[i] = t & (N - 1);
        }
#pragma unroll
        for (int j = 0; j < T; ++j) {
            wA[j] = f2(__ldg(prm.weights + tc[0] + (size_t)N * j), __ldg(prm.weights + tc[2] + (size_t)N * j));
            wB[j] = f2(__ldg(prm.weights + tc[1] + (size_t)N * j), __ldg(prm.weights + tc[3] + (size_t)N * j));
        }
    }
    const int lag0 = lagi[0];
    const bool mixed = lagi[3] != lagi[0];                      // the one quad that straddles the wrap column
    const int64_t R0 = m0 - cq - 1;
    const int row_bytes = N / 4 * 5;
    const uint32_t sh = (uint32_t)((5 * lane) & 3);
    const uint32_t sel = (sh + 3) | ((sh + 2) << 4) | ((sh + 1) << 8) | (sh << 12);
    const uint32_t rd_addr = ring_s + (uint32_t)((5 * lane) >> 2) * 4u;     // W0 of this lane in slot 0
    const uint32_t wr_addr = ring_s + (uint32_t)(lane < 10 ? lane : 0) * 16u;
    const uint32_t is_copier = lane < 10 ? 1u : 0u;

    // valid ring steps: 0 <= R0 + q < rows_in
    const int64_t lo64 = -R0, hi64 = prm.rows_in - R0;
    const int q_lo = (int)max((int64_t)0, min(lo64, (int64_t)0x3fffffff));
    const int q_hi = (int)max((int64_t)0, min(hi64, (int64_t)0x3fffffff));
    const uint8_t *src = wsrc + R0 * (int64_t)row_bytes + (lane < 10 ? lane : 0) * 16;   // ring step 0

    // copy ring step q into `slot` (lanes 0..9 move 16 bytes each; rows outside the batch are zero-filled)
    auto issue = [&](int q, int slot) {
        const uint32_t ok = (q >= q_lo && q < q_hi) ? is_copier : 0u;
        const uint32_t zf = is_copier & ~ok;
        asm volatile(
            "{\n\t.reg .pred p, z;\n\t"
            "setp.ne.u32 p, %2, 0;\n\t"
            "setp.ne.u32 z, %3, 0;\n\t"
            "@p cp.async.cg.shared.global [%0], [%1], 16;\n\t"
            "@z st.shared.v4.u32 [%0], {%4, %4, %4, %4};\n\t"
            "cp.async.commit_group;\n\t}"
            ::"r"(wr_addr + slot * kFirRowBytes), "l"(src), "r"(ok), "r"(zf), "r"(0u) : "memory");
        src += row_bytes;
    };

    __syncwarp();                                               // previous run's reads of the ring are done
#pragma unroll
    for (int k = 0; k < D; ++k) issue(k, k);

    f2 rA[T], rB[T];                                            // sliding window, slot = ring step mod T

    // Protocol: ring steps 0..D-1 are issued up front; at loop step q >= 1, after the warp barrier,
    // ring step q-1+D is issued into the slot ring step q-1 occupied.  At the wait of step q, D+q-1
    // groups have been committed and ring steps <= q must be complete: at most D-2 may be pending.
    auto consume = [&](int q, int slot, int slot_refill, bool refill, f2 &dstA, f2 &dstB) {
        cp_async_wait<D - 2>();
        __syncwarp();                                           // copies visible; last step's reads finished
        if (refill) issue(q - 1 + D, slot_refill);
        uint32_t W0, W1;
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(W0) : "r"(rd_addr + slot * kFirRowBytes) : "memory");
        asm volatile("ld.shared.u32 %0, [%1+4];" : "=r"(W1) : "r"(rd_addr + slot * kFirRowBytes) : "memory");
        float s[4];
        unpack_quad(W0, W1, sel, s);
        dstA = f2(s[0], s[2]);
        dstB = f2(s[1], s[3]);
    };

    // warm-up: ring steps 0 .. T-2
#pragma unroll
    for (int q = 0; q < T - 1; ++q) consume(q, q % D, (q + D - 1) % D, q >= 1, rA[q % T], rB[q % T]);

    // loop step i (0-based) consumes ring step i + T - 1 and completes spectrum  i - 1 + lag  of the run
    const size_t g_stride = (size_t)N * prm.P;                  // next spectrum, same pol (floats)
    float *gp = grow0 + v0 + ((int64_t)lag0 - 1) * (int64_t)g_stride;
    const int n_steps = n_out + 1;

    constexpr int U = (T % D == 0) ? T : (T * D);               // unroll so that both T and D indices are static
    for (int i0 = 0; i0 < n_steps; i0 += U) {
#pragma unroll
        for (int ii = 0; ii < U; ++ii) {
            if (i0 + ii < n_steps) {
                const int q = ii + T - 1;                       // ring step (mod U) consumed now
                consume(i0 + q, q % D, (q + D - 1) % D, true, rA[q % T], rB[q % T]);
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
                const int spec = i0 + ii - 1 + lag0;            // spectrum of the run this window completes
                if (!mixed) {
                    if (spec >= 0 && spec < n_out)
                        stg_stream_f4(reinterpret_cast<float4 *>(gp), make_float4(a0.v.x, a0.v.y, b0.v.x, b0.v.y));
                } else {                                        // columns of this quad belong to two spectra
                    const float gv[4] = {a0.v.x, b0.v.x, a0.v.y, b0.v.y};          // g0, g1, g2, g3
                    const int pos[4] = {0, 2, 1, 3};                                  // stored as (g0, g2, g1, g3)
#pragma unroll
                    for (int cidx = 0; cidx < 4; ++cidx) {
                        const int sp = i0 + ii - 1 + lagi[cidx];
                        if (sp >= 0 && sp < n_out) gp[(int64_t)(lagi[cidx] - lag0) * (int64_t)g_stride + pos[cidx]] = gv[cidx];
                    }
                }
                gp += g_stride;
            }
        }
    }
    cp_async_wait<0>();                                         // drain before the ring is reused
}

template <int T>
__global__ void __launch_bounds__(kFirThreads, 3) fir_kernel(const FirParams prm)
{
    __shared__ __align__(16) unsigned char ring_all[kFirWarps][kFirDepth * kFirRowBytes];
    const int N = 1 << prm.lgN;
    const int stream = blockIdx.z;
    const int a = stream / prm.P, p = stream - a * prm.P;
    const int warp = threadIdx.x >> 5;
    const int v0 = (blockIdx.x * kFirThreads + threadIdx.x) * kFirColsPerThread;
    int64_t m = prm.m_begin + (int64_t)blockIdx.y * prm.rows_per_tile;
    const int64_t m_stop = min(m + (int64_t)prm.rows_per_tile, prm.m_end);
    const uint8_t *sbase = prm.in + (int64_t)stream * prm.stream_bytes;
    const uint8_t *wsrc = sbase + (int64_t)(blockIdx.x * kFirWarps + warp) * kFirRowBytes;
    const int32_t *ctab = prm.coarse + (int64_t)stream * prm.n_coarse;
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(ring_all[warp]);

    while (m < m_stop) {
        const int32_t c = ctab[prm.n_coarse == 1 ? 0 : m];
        int64_t run_end = m_stop;
        if (prm.n_coarse != 1) {
            run_end = m + 1;
            while (run_end < m_stop && ctab[run_end] == c) ++run_end;
        }
        float *grow0 = prm.g + (((int64_t)a * prm.chunk_cap + (m - prm.m_begin)) * prm.P + p) * (int64_t)N;
        fir_run<T>(prm, wsrc, ring_s, (int64_t)c, m, (int)(run_end - m), v0, grow0);
        m = run_end;
    }
}

}  // namespace fe
