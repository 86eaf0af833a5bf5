// fe_fir.cuh -- steps 1-3 of the path: unpack + coarse delay + polyphase FIR (Eq. (1)).
//
// Data layout.  The input of one stream is viewed as a 2-D array of rows of N samples
// ("a 2D array with width 2n, in which the i-th column undergoes a FIR filter").
// A thread owns one 5-byte group = 4 consecutive *input* columns v0..v0+3 and walks down the rows.
// Its 4*T weights stay in registers for the whole tile (PAPER.md:131 keeps them in registers too),
// and so do 4*T partial sums: row r contributes tap j to the spectrum that started j rows earlier,
//     acc[(r - j) mod T] += s[r] * w[j],   j = 0..T-1,
// so every sample is loaded, unpacked and converted exactly once, every tap is one FMA lane-op, and the
// 4*T FMAs of a step are mutually independent (no dot-product dependency chain).  The FMAs are issued
// as packed FFMA2 over the column pairs (0, 2) and (1, 3).
//
// Input staging.  Each warp owns a ring of 16 row segments in shared memory (160 bytes per row:
// 32 lanes x 5 bytes) that it fills with 16-byte cp.async copies in batches of four rows, three
// batches ahead of use, so the HBM/L2 latency is hidden without spending registers and every global
// access is an aligned 128-bit one (BASELINE.json north_star (a)).  Rows outside the batch are
// zero-filled in the ring (R3).
//
// Coarse delay.  With c = N*cq + cr (0 <= cr < N), the sample that Eq. (1)
// pairs with output column t of spectrum m and tap j is row m + j - cq - [t < cr], input column
// v = (t - cr) mod N.  The kernel therefore works in *input* columns (byte-aligned 5-byte groups,
// which is what the paper says pointer arithmetic cannot give for 10-bit samples) and writes the
// row rotated by cr:  g'[v] = g[(v + cr) mod N].  The rotation is undone for free in the
// frequency domain (circular shift theorem): X[k] = exp(-2 pi i k cr / N) * FFT(g')[k], which the
// FFT epilogue folds into the fine-delay phasor.  Columns that wrap (v + cr >= N) read one row
// earlier ("lag"): their partial sums simply belong to the next spectrum, so a lagging thread
// stores one scratch row further down and the inner loop is identical for every lane.  Only the
// warp that holds the single quad straddling the wrap column runs a variant that keeps the previous
// step's result and selects per column.
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
constexpr int kFirBatch = 4;                                        // rows per cp.async group
constexpr int kFirRingBatches = 4;                                  // ring = 4 batches, 3 in flight
constexpr int kFirDepth = kFirBatch * kFirRingBatches;              // 16 ring slots per warp
constexpr int kFirUnroll = 16;                                      // steps per unrolled block (multiple of T and of the ring)

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
    s[2] = (float)((int32_t)(be << 20) >> 22);                  // bits 19..10
    s[3] = (float)((int32_t)(be2 << 22) >> 22);                 // bits  9..0
}

// One chunk of a batch copy: 16 bytes global -> ring, or zeros when the row lies outside the batch.
// ok / zf are 0/1 flags (mutually exclusive; both 0 for lanes that own no chunk).
__device__ __forceinline__ void ring_fill(uint32_t dst, const uint8_t *src, uint32_t ok, uint32_t zf)
{
    asm volatile(
        "{\n\t.reg .pred p, z;\n\t"
        "setp.ne.u32 p, %2, 0;\n\t"
        "setp.ne.u32 z, %3, 0;\n\t"
        "@p cp.async.cg.shared.global [%0], [%1], 16;\n\t"
        "@z st.shared.v4.u32 [%0], {%4, %4, %4, %4};\n\t}"
        ::"r"(dst), "l"(src), "r"(ok), "r"(zf), "r"(0u) : "memory");
}

// One run of n_out consecutive spectra with a constant coarse delay c, for this thread's quad.
//   ring_s    this warp's shared-memory ring, kFirDepth slots of kFirRowBytes
//   wsrc      global address of byte 0 of this warp's 160-byte segment in input row 0 of the stream
//   grow0     scratch row of the run's first spectrum (this stream), column 0
//
// Ring step q holds input row R0 + q, R0 = m0 - cq - 1.  Step q adds tap j of that row to the partial
// sum "mu" = q - 1 - j (relative to the run), which is spectrum mu for a column without lag and
// spectrum mu + 1 for a lagging column.  mu = q - T completes at step q.
template <int T, bool MIXED>
__device__ __forceinline__ void fir_run(const FirParams &prm, const uint8_t *wsrc, uint32_t ring_s, int64_t c,
                                        int64_t m0, int n_out, int v0, float *grow0)
{
    constexpr int U = kFirUnroll;
    static_assert(U % T == 0 && U % kFirDepth == 0, "unroll must cover whole tap and ring periods");
    const int N = 1 << prm.lgN;
    const int lane = threadIdx.x & 31;
    const int cr = (int)(c & (int64_t)(N - 1));
    const int64_t cq = (c - cr) >> prm.lgN;

    // output columns, lag flags and weights of this thread's four input columns
    bool lagc[4];
    f2 wA[T], wB[T];                                            // (col0, col2), (col1, col3)
    {
        int tc[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int t = v0 + i + cr;
            lagc[i] = t >= N;
            tc[i] = t & (N - 1);
        }
#pragma unroll
        for (int j = 0; j < T; ++j) {
            wA[j] = f2(__ldg(prm.weights + tc[0] + (size_t)N * j), __ldg(prm.weights + tc[2] + (size_t)N * j));
            wB[j] = f2(__ldg(prm.weights + tc[1] + (size_t)N * j), __ldg(prm.weights + tc[3] + (size_t)N * j));
        }
    }
    const int lag0 = lagc[0] ? 1 : 0;
    const int64_t R0 = m0 - cq - 1;
    const int row_bytes = N / 4 * 5;
    const uint32_t sh = (uint32_t)((5 * lane) & 3);
    const uint32_t sel = (sh + 3) | ((sh + 2) << 4) | ((sh + 1) << 8) | (sh << 12);
    const uint32_t rd_addr = ring_s + (uint32_t)((5 * lane) >> 2) * 4u;     // W0 of this lane in slot 0

    // Batch copy: 4 rows x 10 chunks of 16 bytes = 40 chunks; lane l moves chunk l, lanes 0..7 also chunk 32+l.
    const int rowA = lane / 10, colA = lane - rowA * 10;
    const int rowB = 3, colB = 2 + lane;
    const bool hasB = lane < 8;
    const uint32_t dstA = ring_s + (uint32_t)(rowA * kFirRowBytes + colA * 16);
    const uint32_t dstB = ring_s + (uint32_t)(rowB * kFirRowBytes + (hasB ? colB : 0) * 16);
    const uint8_t *srcA = wsrc + (R0 + rowA) * (int64_t)row_bytes + colA * 16;
    const uint8_t *srcB = wsrc + (R0 + rowB) * (int64_t)row_bytes + (hasB ? colB : 0) * 16;
    const int64_t batch_bytes = (int64_t)kFirBatch * row_bytes;
    // valid ring steps: 0 <= R0 + q < rows_in  <=>  q_lo <= q < q_lo + span
    const int64_t lo64 = -R0, hi64 = prm.rows_in - R0;
    const int q_lo = (int)max((int64_t)-0x3fffffff, min(lo64, (int64_t)0x3fffffff));
    const int q_hi = (int)max((int64_t)-0x3fffffff, min(hi64, (int64_t)0x3fffffff));
    const uint32_t span = (uint32_t)max(q_hi - q_lo, 0);
    int tA = rowA - q_lo, tB = rowB - q_lo;                     // (row's ring step) - q_lo for the next batch to issue

    auto issue_batch = [&](int slot0) {                         // slot0: first ring slot of the batch (static)
        const uint32_t okA = (uint32_t)tA < span ? 1u : 0u;
        const uint32_t okB = (uint32_t)tB < span ? 1u : 0u;
        ring_fill(dstA + slot0 * kFirRowBytes, srcA, okA, okA ^ 1u);
        ring_fill(dstB + slot0 * kFirRowBytes, srcB, hasB ? okB : 0u, hasB ? (okB ^ 1u) : 0u);
        asm volatile("cp.async.commit_group;" ::: "memory");
        srcA += batch_bytes;
        srcB += batch_bytes;
        tA += kFirBatch;
        tB += kFirBatch;
    };

    __syncwarp();                                               // previous run's reads of the ring are done
#pragma unroll
    for (int b = 0; b < kFirRingBatches - 1; ++b) issue_batch(b * kFirBatch);

    f2 accA[T], accB[T];
#pragma unroll
    for (int j = 0; j < T; ++j) accA[j] = accB[j] = f2(0.f, 0.f);
    float4 prev = make_float4(0.f, 0.f, 0.f, 0.f);

    // scratch pointer of the row stored at step 0 (stores are predicated; see below)
    const size_t g_stride = (size_t)N * prm.P;                  // next spectrum, same pol (floats)
    float *gp = grow0 + v0 + ((int64_t)(MIXED ? 0 : lag0) - T) * (int64_t)g_stride;
    int sp = (MIXED ? 0 : lag0) - T;                            // spectrum (relative to the run) stored at step q

    const int n_steps = n_out + T;
    for (int i0 = 0; i0 < n_steps; i0 += U) {
#pragma unroll
        for (int ii = 0; ii < U; ++ii) {
            if (ii % kFirBatch == 0) {
                // rows of this batch have landed; everyone is done with the previous batch's slots,
                // which the batch issued now overwrites
                cp_async_wait<kFirRingBatches - 2>();
                __syncwarp();
                issue_batch(((ii / kFirBatch + kFirRingBatches - 1) % kFirRingBatches) * kFirBatch);
            }
            const int slot = ii % kFirDepth;
            uint32_t W0, W1;
            asm volatile("ld.shared.u32 %0, [%1];" : "=r"(W0) : "r"(rd_addr + slot * kFirRowBytes) : "memory");
            asm volatile("ld.shared.u32 %0, [%1+4];" : "=r"(W1) : "r"(rd_addr + slot * kFirRowBytes) : "memory");
            float s[4];
            unpack_quad(W0, W1, sel, s);
            const f2 sA(s[0], s[2]), sB(s[1], s[3]);
            accA[ii % T] = sA * wA[0];                           // tap 0 starts partial sum mu = q - 1
            accB[ii % T] = sB * wB[0];
#pragma unroll
            for (int j = 1; j < T; ++j) {
                accA[(ii + T - j) % T] = fma_(sA, wA[j], accA[(ii + T - j) % T]);
                accB[(ii + T - j) % T] = fma_(sB, wB[j], accB[(ii + T - j) % T]);
            }
            const f2 dA = accA[(ii + 1) % T], dB = accB[(ii + 1) % T];     // mu = q - T is complete
            float4 cur = make_float4(dA.v.x, dA.v.y, dB.v.x, dB.v.y);       // (g0, g2, g1, g3)
            if (MIXED) {                                        // lagging columns finished this row one step earlier
                const float4 now = cur;
                cur.x = lagc[0] ? prev.x : now.x;
                cur.y = lagc[2] ? prev.y : now.y;
                cur.z = lagc[1] ? prev.z : now.z;
                cur.w = lagc[3] ? prev.w : now.w;
                prev = now;
            }
            if ((unsigned)sp < (unsigned)n_out) stg_stream_f4(reinterpret_cast<float4 *>(gp), cur);
            gp += g_stride;
            ++sp;
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
        // does this warp hold the quad that straddles the wrap column (v + cr crosses N inside the quad)?
        const int cr = (int)((int64_t)c & (int64_t)(N - 1));
        const bool mixed = (v0 + cr < N) && (v0 + 3 + cr >= N);
        if (__any_sync(0xffffffffu, mixed))
            fir_run<T, true>(prm, wsrc, ring_s, (int64_t)c, m, (int)(run_end - m), v0, grow0);
        else
            fir_run<T, false>(prm, wsrc, ring_s, (int64_t)c, m, (int)(run_end - m), v0, grow0);
        m = run_end;
    }
}

}  // namespace fe
