// fe_fir2.cuh -- steps 1-3 of the path for the pol-packed layout: unpack + coarse delay + polyphase
// FIR (Eq. (1)) of BOTH polarisations of an antenna in one thread.
//
// The two polarisations of an antenna share the weights (one F-engine = the two pols of
// one antenna) and, when their coarse delays are equal, the same column rotation (fe_fir.cuh explains
// the rotation).  A thread then owns one complex FFT input point z[i] = g[2i] + i g[2i+1]
// (PAPER.md:183), i.e. the two input columns 2i, 2i+1, for both pols, and the packed FP32 lanes hold
// (pol 0, pol 1):
//     acc[c][(r - j) mod T] (p0, p1) += s[r][c] (p0, p1) * w[c][j]          (w broadcast to both lanes)
// which halves the weight registers of fe_fir.cuh (2*T instead of 4*T per 64 FMAs) and produces the
// 16-byte unit {Re z p0, Re z p1, Im z p0, Im z p1} that the pol-packed FFT (fe_fft2.cuh) loads with
// one 128-bit access.  Scratch row of (antenna, spectrum): n units = N*2 floats.
//
// Input staging is the ring of fe_fir.cuh with both pols' 80-byte row segments side by side in a
// 160-byte slot.  A 5-byte group (4 samples) is shared by the two threads that own its two points.
#pragma once
#include <cuda_fp16.h>

#include <type_traits>

#include "fe_common.cuh"
#include "fe_fir.cuh"

namespace fe {

struct Fir2Params {
    const uint8_t *in;        // [A][2][stream_bytes]
    const float *weights;     // [N*T]
    float *g;                 // scratch, row a*chunk_cap + (m - m_begin), n units of 16 bytes
    const int32_t *coarse;    // [A*2][n_coarse]; the two pols of an antenna hold equal values
    int64_t n_coarse;
    int64_t stream_bytes;
    int64_t rows_in;
    int64_t m_begin, m_end;
    int64_t chunk_cap;
    int lgN;
    int rows_per_tile;
};

constexpr int kFir2Threads = 128;
constexpr int kFir2Warps = kFir2Threads / 32;

// BITS = sample width of the packed input (10 in the paper's deployment; 4 / 8 / 12 / 16 are its
// bit-depth sweep): same big-endian bit stream, sample u in bits [BITS u, BITS u + BITS).  A warp's
// row segment (64 samples per pol) is 8 BITS bytes, a thread's two samples are 2 BITS bits at bit 2 BITS lane.  The
// geometry of the packed row is the only thing the width changes; arithmetic, partial sums, rotation and the scratch
// layouts are one piece of code (fir2_run).
template <int BITS> struct Fir2Geom {
    static constexpr int seg = 8 * BITS;                              // bytes per warp, row and pol
    static constexpr int slot = 2 * seg;                              // both pols
    static constexpr int cpp = BITS / 2;                              // 16-byte chunks per pol segment
    static constexpr int batch_chunks = 4 * 2 * cpp;                  // kFirBatch rows x 2 pols
    static_assert(BITS == 4 || BITS == 8 || BITS == 10 || BITS == 12 || BITS == 16, "sample width");
    static_assert(batch_chunks <= 64, "at most two chunks per lane and batch");
};
constexpr int kFir2SegBytes = Fir2Geom<10>::seg;                    // 80: 16 groups x 5 bytes
constexpr int kFir2SlotBytes = Fir2Geom<10>::slot;

// Where the finished rows of a run go.  A sink sees, for every step s = 0, 1, .. of the run, one call of
// store(cur) (the 16-byte unit of this thread's point for the run-relative row sp = s - T + lag, which the sink
// counts itself and must ignore outside [0, n_out)), bracketed by before_steps(s) ahead of every 8th step and
// after_steps(s) behind every 8th step (warp-uniform hooks: flow control and completion signalling of the
// pipelined kernel, fe_pipe.cuh; empty here).
struct Fir2ScratchSink {            // two-kernel path: rows of the linear scratch, one row per spectrum
    float *gp;
    size_t g_stride;
    int sp, n_out;
    __device__ __forceinline__ void begin_run(int lag, int T, int n_out_) { gp += ((int64_t)lag - T) * (int64_t)g_stride; sp = lag - T; n_out = n_out_; }
    __device__ __forceinline__ void before_steps(int) {}
    __device__ __forceinline__ void after_steps(int) {}
    __device__ __forceinline__ void end_run() {}
    __device__ __forceinline__ void store(float4 cur)
    {
        asm volatile("{\n\t.reg .pred p;\n\tsetp.lt.u32 p, %5, %6;\n\t@p st.global.v4.f32 [%0], {%1, %2, %3, %4};\n\t}"
                     ::"l"(gp), "f"(cur.x), "f"(cur.y), "f"(cur.z), "f"(cur.w), "r"((unsigned)sp), "r"((unsigned)n_out) : "memory");
        gp += g_stride;
        ++sp;
    }
};

// FP16 scratch (option "scratch_fp16"): the unit is rounded to four halves and stored as 8 bytes
struct Fir2ScratchSinkH16 {
    float *gp;                  // byte address arithmetic in floats: a unit is 2 floats wide, a row N floats
    size_t g_stride;
    int sp, n_out;
    __device__ __forceinline__ void begin_run(int lag, int T, int n_out_) { gp += ((int64_t)lag - T) * (int64_t)g_stride; sp = lag - T; n_out = n_out_; }
    __device__ __forceinline__ void before_steps(int) {}
    __device__ __forceinline__ void after_steps(int) {}
    __device__ __forceinline__ void end_run() {}
    __device__ __forceinline__ void store(float4 cur)
    {
        const __half2 a = __floats2half2_rn(cur.x, cur.y), b = __floats2half2_rn(cur.z, cur.w);
        asm volatile("{\n\t.reg .pred p;\n\tsetp.lt.u32 p, %3, %4;\n\t@p st.global.v2.b32 [%0], {%1, %2};\n\t}"
                     ::"l"(gp), "r"(*reinterpret_cast<const unsigned int *>(&a)), "r"(*reinterpret_cast<const unsigned int *>(&b)),
                       "r"((unsigned)sp), "r"((unsigned)n_out) : "memory");
        gp += g_stride;
        ++sp;
    }
};

// Scratch in the layout of the one-pol FFT (fe_fft.cuh: a row of N floats per (antenna, spectrum, pol), every four
// columns stored as (g0, g2, g1, g3)): point i = 2 q + e holds the columns 4 q + 2 e (Re z, stored at 4 q + e) and
// 4 q + 2 e + 1 (Im z, stored at 4 q + 2 + e); gp points at the pol-0 row, pol 1 is the next row.  Used where the
// pol-packed FFT has no plan (n >= 16384) so that the sweeps of PAPER.md:245 and :273-279 still run a tiled FIR.
struct Fir2OnePolSink {
    float *gp;
    size_t g_stride;
    int N;
    int sp, n_out;
    __device__ __forceinline__ void begin_run(int lag, int T, int n_out_) { gp += ((int64_t)lag - T) * (int64_t)g_stride; sp = lag - T; n_out = n_out_; }
    __device__ __forceinline__ void before_steps(int) {}
    __device__ __forceinline__ void after_steps(int) {}
    __device__ __forceinline__ void end_run() {}
    __device__ __forceinline__ void store(float4 cur)
    {
        asm volatile("{\n\t.reg .pred p;\n\tsetp.lt.u32 p, %6, %7;\n\t@p st.global.f32 [%0], %2;\n\t@p st.global.f32 [%0+8], %4;\n\t"
                     "@p st.global.f32 [%1], %3;\n\t@p st.global.f32 [%1+8], %5;\n\t}"
                     ::"l"(gp), "l"(gp + N), "f"(cur.x), "f"(cur.y), "f"(cur.z), "f"(cur.w), "r"((unsigned)sp), "r"((unsigned)n_out) : "memory");
        gp += g_stride;
        ++sp;
    }
};

// Ring step q holds input row R0 + q of both pols, R0 = m0 - cq - 1; see fir_run in fe_fir.cuh for the
// partial-sum bookkeeping, which is identical.
// NC: the row width N when the caller knows it at compile time (row strides become immediates), else 0.
template <int T, bool MIXED, class Sink, int NC = 0, int BITS = 10>
__device__ __forceinline__ void fir2_run(const Fir2Params &prm, const uint8_t *wsrc, uint32_t ring_s, int64_t c,
                                         int64_t m0, int n_out, int i_pt, Sink &sink)
{
    using G = Fir2Geom<BITS>;
    constexpr int U = kFirUnroll;
    static_assert(U % T == 0 && U % kFirDepth == 0, "unroll must cover whole tap and ring periods");
    const int N = NC ? NC : 1 << prm.lgN;
    const int lane = threadIdx.x & 31;
    const int cr = (int)(c & (int64_t)(N - 1));
    const int64_t cq = (c - cr) >> prm.lgN;
    const int v0 = 2 * i_pt;                                    // input columns v0 (Re z), v0 + 1 (Im z)

    bool lagc[2];
    float w0[T], w1[T];
    {
        int tc[2];
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const int t = v0 + i + cr;
            lagc[i] = t >= N;
            tc[i] = t & (N - 1);
        }
#pragma unroll
        for (int j = 0; j < T; ++j) {
            w0[j] = __ldg(prm.weights + tc[0] + (size_t)N * j);
            w1[j] = __ldg(prm.weights + tc[1] + (size_t)N * j);
        }
    }
    const int lag0 = lagc[0] ? 1 : 0;
    const int64_t R0 = m0 - cq - 1;
    const int row_bytes = N / 8 * BITS;

    // this thread's bits in a slot: 2 BITS bits at bit 2 BITS lane of the warp's segment; b0..b3 = the four bytes
    // that start at byte boff, after sha leading bits (sha + 2 BITS <= 32 for every supported width)
    const uint32_t bit0 = 2u * BITS * (uint32_t)lane;
    const uint32_t boff = bit0 >> 3;
    const uint32_t sh = boff & 3;
    const uint32_t sel = (sh + 3) | ((sh + 2) << 4) | ((sh + 1) << 8) | (sh << 12);
    const uint32_t rd_addr = ring_s + (boff >> 2) * 4u;          // W0 of pol 0 in slot 0
    const uint32_t sha = bit0 & 7u;                              // left shift that brings sample a to the top bits

    // Batch copy: 4 rows x 2 pols x cpp chunks of 16 bytes; lane l moves chunk l and, where it exists, chunk 32 + l.
    const int idxA = lane, idxB = 32 + lane;
    const bool hasA = idxA < G::batch_chunks, hasB = idxB < G::batch_chunks;
    const int rowA = hasA ? idxA / (2 * G::cpp) : 0, remA = hasA ? idxA % (2 * G::cpp) : 0, polA = remA / G::cpp, colA = remA % G::cpp;
    const int rowB = hasB ? idxB / (2 * G::cpp) : 0, remB = hasB ? idxB % (2 * G::cpp) : 0, polB = remB / G::cpp, colB = remB % G::cpp;
    const uint32_t dstA = ring_s + (uint32_t)(rowA * G::slot + polA * G::seg + colA * 16);
    const uint32_t dstB = ring_s + (uint32_t)(rowB * G::slot + polB * G::seg + colB * 16);
    const uint8_t *srcA = wsrc + polA * prm.stream_bytes + (R0 + rowA) * (int64_t)row_bytes + colA * 16;
    const uint8_t *srcB = wsrc + polB * prm.stream_bytes + (R0 + rowB) * (int64_t)row_bytes + colB * 16;
    const int64_t batch_bytes = (int64_t)kFirBatch * row_bytes;
    const int64_t lo64 = -R0, hi64 = prm.rows_in - R0;
    const int q_lo = (int)max((int64_t)-0x3fffffff, min(lo64, (int64_t)0x3fffffff));
    const int q_hi = (int)max((int64_t)-0x3fffffff, min(hi64, (int64_t)0x3fffffff));
    const uint32_t span = (uint32_t)max(q_hi - q_lo, 0);
    int tA = rowA - q_lo, tB = rowB - q_lo;

    auto issue_batch = [&](int slot0) {
        const uint32_t okA = (uint32_t)tA < span ? 1u : 0u;
        const uint32_t okB = (uint32_t)tB < span ? 1u : 0u;
        ring_fill(dstA + slot0 * G::slot, srcA, hasA ? okA : 0u, hasA ? (okA ^ 1u) : 0u);
        ring_fill(dstB + slot0 * G::slot, srcB, hasB ? okB : 0u, hasB ? (okB ^ 1u) : 0u);
        asm volatile("cp.async.commit_group;" ::: "memory");
        srcA += batch_bytes;
        srcB += batch_bytes;
        tA += kFirBatch;
        tB += kFirBatch;
    };

    __syncwarp();
#pragma unroll
    for (int b = 0; b < kFirRingBatches - 1; ++b) issue_batch(b * kFirBatch);

    f2 acc0[T], acc1[T];                                        // columns v0, v0+1; lanes (pol 0, pol 1)
#pragma unroll
    for (int j = 0; j < T; ++j) acc0[j] = acc1[j] = f2(0.f, 0.f);
    float4 prev = make_float4(0.f, 0.f, 0.f, 0.f);

    sink.begin_run(MIXED ? 0 : lag0, T, n_out);

    // The loop is software-pipelined by one step and has no branch in its unrolled body: the raw words of step
    // ii + 1 are read from the ring while the FMAs of step ii issue, and the scratch store is a predicated
    // instruction, so the unpack chain (LDS -> PRMT -> SHF -> I2FP) of the next step hides behind 32 FFMA2s.
    auto load_raw = [&](int slot, uint32_t (&raw)[4]) {
        const uint32_t ad = rd_addr + slot * G::slot;
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(raw[0]) : "r"(ad) : "memory");
        asm volatile("ld.shared.u32 %0, [%1+4];" : "=r"(raw[1]) : "r"(ad) : "memory");
        asm volatile("ld.shared.u32 %0, [%1+%2];" : "=r"(raw[2]) : "r"(ad), "n"(G::seg) : "memory");
        asm volatile("ld.shared.u32 %0, [%1+%2];" : "=r"(raw[3]) : "r"(ad), "n"(G::seg + 4) : "memory");
    };
    uint32_t nxt[4];
    cp_async_wait<kFirRingBatches - 2>();
    __syncwarp();
    issue_batch((kFirRingBatches - 1) * kFirBatch);
    load_raw(0, nxt);

    const int n_steps = n_out + T;
    for (int i0 = 0; i0 < n_steps; i0 += U) {
#pragma unroll
        for (int ii = 0; ii < U; ++ii) {
            if (ii % 8 == 0) sink.before_steps(i0 + ii);
            const uint32_t P0a = nxt[0], P0b = nxt[1], P1a = nxt[2], P1b = nxt[3];
            if ((ii + 1) % kFirBatch == 0) {
                // the batch that holds step ii + 1 has landed; every lane holds the words of step ii, so the batch
                // issued now may overwrite the slots of steps ii - 3 .. ii
                cp_async_wait<kFirRingBatches - 2>();
                __syncwarp();
                issue_batch((((ii + 1) / kFirBatch + kFirRingBatches - 1) % kFirRingBatches) * kFirBatch);
            }
            load_raw((ii + 1) % kFirDepth, nxt);
            const uint32_t be0 = __byte_perm(P0a, P0b, sel) << sha;     // sample a in the top BITS bits, b below it
            const uint32_t be1 = __byte_perm(P1a, P1b, sel) << sha;
            const f2 s0((float)((int32_t)be0 >> (32 - BITS)), (float)((int32_t)be1 >> (32 - BITS)));                    // column v0, (p0, p1)
            const f2 s1((float)((int32_t)(be0 << BITS) >> (32 - BITS)), (float)((int32_t)(be1 << BITS) >> (32 - BITS)));  // column v0 + 1
            // one column at a time: consecutive FFMA2s then share the sample operand, which ptxas keeps in the
            // operand-reuse cache (a FFMA2 with three fresh register operands issues at ~77 % of the packed rate,
            // measured; with the sample reused it issues at ~96 %)
            acc0[ii % T] = s0 * w0[0];
#pragma unroll
            for (int j = 1; j < T; ++j) acc0[(ii + T - j) % T] = fma_(s0, w0[j], acc0[(ii + T - j) % T]);
            acc1[ii % T] = s1 * w1[0];
#pragma unroll
            for (int j = 1; j < T; ++j) acc1[(ii + T - j) % T] = fma_(s1, w1[j], acc1[(ii + T - j) % T]);
            const f2 d0 = acc0[(ii + 1) % T], d1 = acc1[(ii + 1) % T];
            float4 cur = make_float4(d0.v.x, d0.v.y, d1.v.x, d1.v.y);       // {Re p0, Re p1, Im p0, Im p1}
            if (MIXED) {
                const float4 now = cur;
                cur.x = lagc[0] ? prev.x : now.x;
                cur.y = lagc[0] ? prev.y : now.y;
                cur.z = lagc[1] ? prev.z : now.z;
                cur.w = lagc[1] ? prev.w : now.w;
                prev = now;
            }
            sink.store(cur);
            if (ii % 8 == 7) sink.after_steps(i0 + ii);
        }
    }
    cp_async_wait<0>();
    sink.end_run();
}

// OUT: where the finished rows go
enum { kFir2OutPacked = 0, kFir2OutPackedH16 = 1, kFir2OutOnePol = 2 };

template <int T, int OUT = kFir2OutPacked, int BITS = 10>
__global__ void __launch_bounds__(kFir2Threads, 4) fir2_kernel(const Fir2Params prm)
{
    using G = Fir2Geom<BITS>;
    // +16: the second word of the last lane's pol-1 group may lie just past the last slot (never selected)
    __shared__ __align__(16) unsigned char ring_all[kFir2Warps * kFirDepth * G::slot + 16];
    const int N = 1 << prm.lgN;
    const int a = blockIdx.z;
    const int warp = threadIdx.x >> 5;
    const int i_pt = blockIdx.x * kFir2Threads + threadIdx.x;   // complex point index 0..n-1
    int64_t m = prm.m_begin + (int64_t)blockIdx.y * prm.rows_per_tile;
    const int64_t m_stop = min(m + (int64_t)prm.rows_per_tile, prm.m_end);
    const uint8_t *sbase = prm.in + (int64_t)a * 2 * prm.stream_bytes;
    const uint8_t *wsrc = sbase + (int64_t)(blockIdx.x * kFir2Warps + warp) * G::seg;
    const int32_t *ctab = prm.coarse + (int64_t)a * 2 * prm.n_coarse;
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(ring_all + warp * kFirDepth * G::slot);

    while (m < m_stop) {
        const int32_t c = ctab[prm.n_coarse == 1 ? 0 : m];
        int64_t run_end = m_stop;
        if (prm.n_coarse != 1) {
            run_end = m + 1;
            while (run_end < m_stop && ctab[run_end] == c) ++run_end;
        }
        const int cr = (int)((int64_t)c & (int64_t)(N - 1));
        const bool mixed = (2 * i_pt + cr < N) && (2 * i_pt + 1 + cr >= N);
        const int n_run = (int)(run_end - m);
        const int64_t row = (int64_t)a * prm.chunk_cap + (m - prm.m_begin);
        auto run = [&](auto &sink) {
            if (__any_sync(0xffffffffu, mixed))
                fir2_run<T, true, std::remove_reference_t<decltype(sink)>, 0, BITS>(prm, wsrc, ring_s, (int64_t)c, m, n_run, i_pt, sink);
            else
                fir2_run<T, false, std::remove_reference_t<decltype(sink)>, 0, BITS>(prm, wsrc, ring_s, (int64_t)c, m, n_run, i_pt, sink);
        };
        if constexpr (OUT == kFir2OutPackedH16) {               // 8-byte units: a row is N floats wide
            Fir2ScratchSinkH16 sink{prm.g + row * (int64_t)N + 2 * i_pt, (size_t)N, 0, 0};
            run(sink);
        } else if constexpr (OUT == kFir2OutOnePol) {           // rows (antenna, spectrum, pol) of N floats
            Fir2OnePolSink sink{prm.g + row * (int64_t)N * 2 + 4 * (i_pt >> 1) + (i_pt & 1), (size_t)N * 2, N, 0, 0};
            run(sink);
        } else {
            Fir2ScratchSink sink{prm.g + row * (int64_t)N * 2 + 4 * i_pt, (size_t)N * 2, 0, 0};
            run(sink);
        }
        m = run_end;
    }
}

}  // namespace fe
