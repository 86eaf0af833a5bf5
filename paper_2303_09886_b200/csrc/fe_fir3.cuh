// fe_fir3.cuh -- steps 1-3 of the path for the pol-packed layout, ONE input column per thread (used for T = 32).
//
// Same arithmetic and same scratch layout as fe_fir2.cuh (unit {Re z p0, Re z p1, Im z p0, Im z p1}, z[i] =
// g'[2i] + i g'[2i+1], row rotated by c mod N), but a thread owns a single column v of both pols:
//     acc[(r - j) mod T] (p0, p1) += s[r][v] (p0, p1) * w[v][j]
// T weights + T packed partial sums = 3T registers instead of 6T, which is what lets 32 taps
// stay in registers.  (For T <= 16 the two-column kernel is as fast: both are bound by the scratch writes.)
// All T FFMA2s of a step share the sample operand (operand-reuse cache), and a thread's column either lags or
// does not, so there is no mixed-lag variant.
//
// Input staging: one ring of 16 rows per CTA, 160 bytes (128 columns) per pol and row, filled by 16-byte
// cp.async copies in batches of four rows; 80 of the 128 threads move one chunk per batch.
#pragma once
#include "fe_common.cuh"
#include "fe_fir.cuh"
#include "fe_fir2.cuh"

namespace fe {

constexpr int kFir3Threads = 128;
constexpr int kFir3SegBytes = 160;                                  // 128 columns x 10 bits
constexpr int kFir3SlotBytes = 2 * kFir3SegBytes;                   // both pols
constexpr int kFir3RingBytes = kFirDepth * kFir3SlotBytes + 16;     // +16: the second word of the last thread's group

// ONEPOL: write the scratch in the layout of the one-pol FFT (fe_fft.cuh: a row of N floats per (antenna, spectrum,
// pol), every four columns stored as (g0, g2, g1, g3)) instead of the pol-packed units, so that shapes the pol-packed
// FFT does not cover (n >= 16384) still get a tiled FIR for 32 taps (Fig. 8: "for 32 768 channels").
template <int T, bool ONEPOL = false>
__device__ __forceinline__ void fir3_run(const Fir2Params &prm, const uint8_t *csrc, uint32_t ring_s, int64_t c,
                                         int64_t m0, int n_out, int v, float *grow0)
{
    constexpr int U = T > kFirUnroll ? T : kFirUnroll;
    static_assert(U % T == 0 && U % kFirDepth == 0, "unroll must cover whole tap and ring periods");
    const int N = 1 << prm.lgN;
    const int tid = threadIdx.x;
    const int cr = (int)(c & (int64_t)(N - 1));
    const int64_t cq = (c - cr) >> prm.lgN;

    const int t_out = v + cr;
    const int lag = t_out >= N ? 1 : 0;
    float w[T];
#pragma unroll
    for (int j = 0; j < T; ++j) w[j] = __ldg(prm.weights + (t_out & (N - 1)) + (size_t)N * j);

    const int64_t R0 = m0 - cq - 1;
    const int row_bytes = N / 4 * 5;

    // this thread's 10 bits: group tid / 4, sample r = tid % 4: bytes [5 g + r, 5 g + r + 2), field at bit 6 - 2 r
    const int r4 = tid & 3;
    const uint32_t boff = (uint32_t)(5 * (tid >> 2) + r4);
    const uint32_t sh = boff & 3;
    const uint32_t sel = (sh + 1) << 8 | sh << 12;                // bytes [boff], [boff + 1] -> bits 31..16 (big endian)
    const uint32_t rd_addr = ring_s + (boff >> 2) * 4u;           // aligned word that holds byte boff, pol 0, slot 0
    const uint32_t shl = 2u * (uint32_t)r4;                       // brings the field's MSB to bit 31

    // batch copy: 4 rows x 2 pols x 10 chunks of 16 bytes = 80 chunks, one per thread tid < 80
    const bool mover = tid < 80;
    const int rowA = tid / 20, remA = tid - rowA * 20, polA = remA / 10, colA = remA - polA * 10;
    const uint32_t dstA = ring_s + (uint32_t)((mover ? rowA : 0) * kFir3SlotBytes + (mover ? polA : 0) * kFir3SegBytes + (mover ? colA : 0) * 16);
    const uint8_t *srcA = csrc + (mover ? polA : 0) * prm.stream_bytes + (R0 + (mover ? rowA : 0)) * (int64_t)row_bytes + (mover ? colA : 0) * 16;
    const int64_t batch_bytes = (int64_t)kFirBatch * row_bytes;
    const int64_t lo64 = -R0, hi64 = prm.rows_in - R0;
    const int q_lo = (int)max((int64_t)-0x3fffffff, min(lo64, (int64_t)0x3fffffff));
    const int q_hi = (int)max((int64_t)-0x3fffffff, min(hi64, (int64_t)0x3fffffff));
    const uint32_t span = (uint32_t)max(q_hi - q_lo, 0);
    int tA = rowA - q_lo;

    auto issue_batch = [&](int slot0) {
        const uint32_t okA = (uint32_t)tA < span ? 1u : 0u;
        ring_fill(dstA + slot0 * kFir3SlotBytes, srcA, mover ? okA : 0u, mover ? (okA ^ 1u) : 0u);
        asm volatile("cp.async.commit_group;" ::: "memory");
        srcA += batch_bytes;
        tA += kFirBatch;
    };
    auto load_raw = [&](int slot, uint32_t (&raw)[4]) {
        const uint32_t ad = rd_addr + slot * kFir3SlotBytes;
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(raw[0]) : "r"(ad) : "memory");
        asm volatile("ld.shared.u32 %0, [%1+4];" : "=r"(raw[1]) : "r"(ad) : "memory");
        asm volatile("ld.shared.u32 %0, [%1+160];" : "=r"(raw[2]) : "r"(ad) : "memory");
        asm volatile("ld.shared.u32 %0, [%1+164];" : "=r"(raw[3]) : "r"(ad) : "memory");
    };

    __syncthreads();                                              // the previous run is done with the ring
#pragma unroll
    for (int b = 0; b < kFirRingBatches - 1; ++b) issue_batch(b * kFirBatch);

    f2 acc[T];
#pragma unroll
    for (int j = 0; j < T; ++j) acc[j] = f2(0.f, 0.f);

    const size_t g_stride = (size_t)N * 2;                        // next spectrum (floats)
    // ONEPOL: grow0 is row (antenna, spectrum, pol 0); pol 1 is the next row; column v sits at 4 (v / 4) + {0, 2, 1, 3}[v % 4]
    float *gp = grow0 + (ONEPOL ? 4 * (v >> 2) + (((v & 1) << 1) | ((v >> 1) & 1)) : 4 * (v >> 1) + 2 * (v & 1)) +
                ((int64_t)lag - T) * (int64_t)g_stride;
    int sp = lag - T;

    uint32_t nxt[4];
    cp_async_wait<kFirRingBatches - 2>();
    __syncthreads();
    issue_batch((kFirRingBatches - 1) * kFirBatch);
    load_raw(0, nxt);

    const int n_steps = n_out + T;
    for (int i0 = 0; i0 < n_steps; i0 += U) {
#pragma unroll
        for (int ii = 0; ii < U; ++ii) {
            const uint32_t P0a = nxt[0], P0b = nxt[1], P1a = nxt[2], P1b = nxt[3];
            if ((ii + 1) % kFirBatch == 0) {
                cp_async_wait<kFirRingBatches - 2>();
                __syncthreads();
                issue_batch(((((ii + 1) / kFirBatch) + kFirRingBatches - 1) % kFirRingBatches) * kFirBatch);
            }
            load_raw((ii + 1) % kFirDepth, nxt);
            const int32_t x0 = (int32_t)(__byte_perm(P0a, P0b, sel) << shl) >> 22;
            const int32_t x1 = (int32_t)(__byte_perm(P1a, P1b, sel) << shl) >> 22;
            const f2 s((float)x0, (float)x1);                     // (pol 0, pol 1)
            acc[ii % T] = s * w[0];
#pragma unroll
            for (int j = 1; j < T; ++j) acc[(ii + T - j) % T] = fma_(s, w[j], acc[(ii + T - j) % T]);
            const f2 d = acc[(ii + 1) % T];
            if (ONEPOL)
                asm volatile("{\n\t.reg .pred p;\n\tsetp.lt.u32 p, %4, %5;\n\t@p st.global.f32 [%0], %2;\n\t@p st.global.f32 [%1], %3;\n\t}"
                             ::"l"(gp), "l"(gp + N), "f"(d.v.x), "f"(d.v.y), "r"((unsigned)sp), "r"((unsigned)n_out) : "memory");
            else
                asm volatile("{\n\t.reg .pred p;\n\tsetp.lt.u32 p, %3, %4;\n\t@p st.global.v2.f32 [%0], {%1, %2};\n\t}"
                             ::"l"(gp), "f"(d.v.x), "f"(d.v.y), "r"((unsigned)sp), "r"((unsigned)n_out) : "memory");
            gp += g_stride;
            ++sp;
        }
    }
    cp_async_wait<0>();
}

template <int T, bool ONEPOL = false>
__global__ void __launch_bounds__(kFir3Threads, 4) fir3_kernel(const Fir2Params prm)
{
    __shared__ __align__(16) unsigned char ring_all[kFir3RingBytes];
    const int N = 1 << prm.lgN;
    const int a = blockIdx.z;
    const int v = blockIdx.x * kFir3Threads + threadIdx.x;        // input column 0..N-1
    int64_t m = prm.m_begin + (int64_t)blockIdx.y * prm.rows_per_tile;
    const int64_t m_stop = min(m + (int64_t)prm.rows_per_tile, prm.m_end);
    const uint8_t *csrc = prm.in + (int64_t)a * 2 * prm.stream_bytes + (int64_t)blockIdx.x * kFir3SegBytes;
    const int32_t *ctab = prm.coarse + (int64_t)a * 2 * prm.n_coarse;
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(ring_all);

    while (m < m_stop) {
        const int32_t c = ctab[prm.n_coarse == 1 ? 0 : m];
        int64_t run_end = m_stop;
        if (prm.n_coarse != 1) {
            run_end = m + 1;
            while (run_end < m_stop && ctab[run_end] == c) ++run_end;
        }
        float *grow0 = prm.g + ((int64_t)a * prm.chunk_cap + (m - prm.m_begin)) * (int64_t)N * 2;
        fir3_run<T, ONEPOL>(prm, csrc, ring_s, (int64_t)c, m, (int)(run_end - m), v, grow0);
        m = run_end;
    }
}

}  // namespace fe
