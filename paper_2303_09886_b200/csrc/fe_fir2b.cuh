// fe_fir2b.cuh -- the pol-packed FIR of fe_fir2.cuh for input sample widths other than 10 bits.
//
// The paper sweeps the input bit depth over 4, 8, 12 and 16 bits.  The arithmetic, the partial-sum
// bookkeeping, the coarse-delay rotation and the scratch layout are those of fe_fir2.cuh; only the geometry of the
// packed row changes (bytes per warp segment, chunks per batch copy, position and width of a thread's two samples).
// It is a separate copy so that the 10-bit kernel of the headline path keeps its exact instruction stream.
#pragma once
#include "fe_common.cuh"
#include "fe_fir.cuh"
#include "fe_fir2.cuh"

namespace fe {

// BITS = sample width of the packed input (10 in the paper's deployment; 4 / 8 / 12 / 16 are its
// bit-depth sweep): same big-endian bit stream, sample u in bits [BITS u, BITS u + BITS).  A warp's
// row segment (64 samples per pol) is 8 BITS bytes, a thread's two samples are 2 BITS bits at bit 2 BITS lane.
template <int BITS> struct Fir2Geom {
    static constexpr int seg = 8 * BITS;                              // bytes per warp, row and pol
    static constexpr int slot = 2 * seg;                              // both pols
    static constexpr int cpp = BITS / 2;                              // 16-byte chunks per pol segment
    static constexpr int batch_chunks = kFirBatch * 2 * cpp;          // 4 rows x 2 pols
    static_assert(BITS == 4 || BITS == 8 || BITS == 10 || BITS == 12 || BITS == 16, "sample width");
    static_assert(batch_chunks <= 64, "at most two chunks per lane and batch");
};

// ONEPOL: write the scratch in the layout of the one-pol FFT (fe_fft.cuh: a row of N floats per (antenna, spectrum,
// pol), every four columns stored as (g0, g2, g1, g3)) instead of the pol-packed units: the bit-depth sweep at
// n = 32768 (Fig. 11), which the pol-packed FFT does not cover, then still runs a tiled FIR.
template <int T, bool MIXED, int BITS, bool ONEPOL = false>
__device__ __forceinline__ void fir2b_run(const Fir2Params &prm, const uint8_t *wsrc, uint32_t ring_s, int64_t c,
                                         int64_t m0, int n_out, int i_pt, float *grow0)
{
    using G = Fir2Geom<BITS>;
    constexpr int U = kFirUnroll;
    static_assert(U % T == 0 && U % kFirDepth == 0, "unroll must cover whole tap and ring periods");
    const int N = 1 << prm.lgN;
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

    // this thread's two samples: 2 BITS bits at bit 2 BITS lane of the warp's segment, i.e. inside the four bytes
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

    const size_t g_stride = (size_t)N * 2;                      // next spectrum (floats): n units of 4 floats
    // ONEPOL: grow0 is row (antenna, spectrum, pol 0), pol 1 the next row; point i = 2 q + e holds the columns
    // 4 q + 2 e (Re z, stored at 4 q + e) and 4 q + 2 e + 1 (Im z, stored at 4 q + 2 + e)
    float *gp = grow0 + (ONEPOL ? 4 * (i_pt >> 1) + (i_pt & 1) : 4 * i_pt) + ((int64_t)(MIXED ? 0 : lag0) - T) * (int64_t)g_stride;
    int sp = (MIXED ? 0 : lag0) - T;

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
            const f2 s0((float)((int32_t)be0 >> (32 - BITS)), (float)((int32_t)be1 >> (32 - BITS)));          // column v0, (p0, p1)
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
            if (ONEPOL)
                asm volatile("{\n\t.reg .pred p;\n\tsetp.lt.u32 p, %6, %7;\n\t@p st.global.f32 [%0], %2;\n\t@p st.global.f32 [%0+8], %4;\n\t"
                             "@p st.global.f32 [%1], %3;\n\t@p st.global.f32 [%1+8], %5;\n\t}"
                             ::"l"(gp), "l"(gp + N), "f"(cur.x), "f"(cur.y), "f"(cur.z), "f"(cur.w), "r"((unsigned)sp), "r"((unsigned)n_out) : "memory");
            else
                asm volatile("{\n\t.reg .pred p;\n\tsetp.lt.u32 p, %5, %6;\n\t@p st.global.v4.f32 [%0], {%1, %2, %3, %4};\n\t}"
                             ::"l"(gp), "f"(cur.x), "f"(cur.y), "f"(cur.z), "f"(cur.w), "r"((unsigned)sp), "r"((unsigned)n_out) : "memory");
            gp += g_stride;
            ++sp;
        }
    }
    cp_async_wait<0>();
}

template <int T, int BITS, bool ONEPOL = false>
__global__ void __launch_bounds__(kFir2Threads, 4) fir2b_kernel(const Fir2Params prm)
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
        float *grow0 = prm.g + ((int64_t)a * prm.chunk_cap + (m - prm.m_begin)) * (int64_t)N * 2;
        const int cr = (int)((int64_t)c & (int64_t)(N - 1));
        const bool mixed = (2 * i_pt + cr < N) && (2 * i_pt + 1 + cr >= N);
        if (__any_sync(0xffffffffu, mixed))
            fir2b_run<T, true, BITS, ONEPOL>(prm, wsrc, ring_s, (int64_t)c, m, (int)(run_end - m), i_pt, grow0);
        else
            fir2b_run<T, false, BITS, ONEPOL>(prm, wsrc, ring_s, (int64_t)c, m, (int)(run_end - m), i_pt, grow0);
        m = run_end;
    }
}

}  // namespace fe
