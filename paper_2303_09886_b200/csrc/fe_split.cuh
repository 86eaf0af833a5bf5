// fe_split.cuh -- the pol-packed path split the way the paper's conclusion proposes ("step 2 of the
// six-step FFT merged into the PFB FIR kernel"): the n-point complex transform of a spectrum is n = 16 M,
//
//   stage 1 (producer, with the FIR)   y[ka][i'] = W_n^{i' ka} * sum_{q < 16} z[i' + M q] W_16^{q ka}         (ka < 16, i' < M)
//   stage 2 (consumer)                 Z[ka + 16 k'] = sum_{i' < M} y[ka][i'] W_M^{i' k'}                     (k' < M)
//
// i.e. decimation in frequency with the first digit of radix 16.  Stage 1 only needs the 16 points {i' + M q} of a
// row, so a CTA that runs the polyphase FIR (Eq. (1)) on the columns of 16 consecutive i' and all q
// owns complete butterflies: its FIR warps put finished rows into a shared-memory tile, its butterfly warps take them
// out again 16 at a time, and what goes to the next stage is y, laid out [antenna][spectrum][ka][i'].
// Stage 2 is then 16 independent M-point transforms per spectrum, and the real-FFT post-twiddle of PAPER.md:183 couples
// exactly the transforms ka and 16 - ka (a channel k and its mirror n - k):
//   M = 256 (n = 4096)          ONE WARP does the pair, 16 points x 2 pols per thread, warp-level synchronisation
//                               only: radix 16, exchange through the warp's own 8.5 KB of shared memory, radix 16, mirror
//                               exchange, then post-twiddle, fine-delay rotation, gain and
//                               quantisation in registers; the int8 words of a spectrum are collected
//                               in a staging row per CTA so that the global stores are full 128-byte lines;
//   M = 1024, 2048 (n >= 16384)  one CTA of two teams does the pair with the pol-packed M-point plan of fe_fft2.cuh
//                               (split_pair_kernel, further down).
// Measured: the default for n >= 16384 (config 3: 116 -> 158 Gsample/s); at n = 4096 the
// consumer is faster than the one-CTA-per-spectrum FFT but the producer, with a third of the butterflies next to the
// FIR, is FMA-issue bound, and the two-kernel path of fe_fir2.cuh / fe_fft2.cuh stays the default there.
#pragma once
#include "fe_common.cuh"
#include "fe_fft.cuh"
#include "fe_fft2.cuh"
#include "fe_fir2.cuh"

namespace fe {

constexpr int kSubM = 256;                          // points of a stage-2 transform
constexpr int kSplitFirWarps = 8;                   // 256 complex points per producer CTA
constexpr int kSplitBfWarps = 4;
constexpr int kSplitProducerThreads = 32 * (kSplitFirWarps + kSplitBfWarps);
constexpr int kSplitTileSlots = 16;                 // rows of the tile: two blocks of eight steps
constexpr int kSplitTileBytes = kSplitTileSlots * 256 * 16;
constexpr int kSplitRingBytes = kFirDepth * kFir2SlotBytes + 16;
constexpr int kXHalf = 16 * 17;                     // units of one transform's exchange buffer (rows skewed by one unit)
constexpr int kStagePitch = 258;                    // words per ka row of the staging buffer (banks: 2 ka + k')

struct SplitParams {
    Fir2Params fir;           // in, weights, g (= y), coarse, n_coarse, stream_bytes, rows_in, m_begin, m_end, chunk_cap, lgN, rows_per_tile
    Fft2Params fft;           // g (= y), out, out_f32, tpost, rg2, coarse, fine_d, fine_phi, n_coarse, n_fine, m_begin, m_end, chunk_cap, n_spectra, per_spectrum
    const float2 *tw1;        // [K1][M]    W_n^{ka i'}     (cos, -sin); M = n / K1 points per stage-2 transform
    const float2 *ptw1, *ptw2;  // M > 256: pass twiddles of the M-point plan of the pair kernel (fe_fft2.cuh layout)
    const float2 *tw256;      // [16][16]   W_256^{kb t}
};

// ---------------------------------------------------------------------------------------------------------------
// producer: FIR warps
// ---------------------------------------------------------------------------------------------------------------
template <int CB>
__device__ __forceinline__ void ring_fill_n(uint32_t dst, const uint8_t *src, uint32_t src_bytes)
{
    // src_bytes = CB copies, 0 zero-fills (rows outside the batch, R3); the source is not read then
    if constexpr (CB == 16)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
    else if constexpr (CB == 8)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}

__device__ __forceinline__ void sts_f4(uint32_t saddr, float4 v)
{
    asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(saddr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

// One run of n_out consecutive spectra with a constant coarse delay c for this warp's 32 points: the loop of
// fir2_run (fe_fir2.cuh; partial sums, ring, unpack are identical) with two differences.
//   * The warp's points are NP runs of 32 / NP consecutive points (IL = 256 / K1 consecutive i' per q), so a ring
//     slot is filled by 16 / NP-byte copies from NP places of the row; the slot layout and the unpack do not change.
//   * Every lane is aligned to the same spectrum: a column that wraps (lag) hands over the previous step's value,
//     so that step s finishes row s - T of the run on every lane and the row goes to tile slot s mod 16.
// Blocks of eight steps are handed to the butterfly warps through full / empty mbarriers; gx counts the blocks of
// this CTA since its start (buffer gx & 1, phase gx >> 1).
template <int T, int IL, int M>
__device__ __forceinline__ void split_fir_run(const Fir2Params &prm, const uint8_t *abase, int i0, int fw, uint32_t ring_s,
                                              int64_t c, int64_t m0, int n_out, uint32_t tile_thr, uint32_t full0,
                                              uint32_t empty0, unsigned &gx)
{
    constexpr int U = kFirUnroll;
    static_assert(U % T == 0 && U == kFirDepth && U == kSplitTileSlots, "unroll = ring depth = tile slots");
    constexpr int NP = IL >= 32 ? 1 : 32 / IL;                  // pieces per warp, row and pol
    constexpr int CB = 16 / NP;                                 // bytes per copy (5 copies per piece)
    constexpr int NCH = 40 * NP, NT = (NCH + 31) / 32;          // copies per batch of 4 rows, per lane
    const int N = 1 << prm.lgN;
    const int lane = threadIdx.x & 31;
    const int pt = 32 * fw + lane;                              // point of the CTA: q = pt / IL, il = pt % IL
    const int i_pt = i0 + (pt % IL) + M * (pt / IL);
    const int cr = (int)(c & (int64_t)(N - 1));
    const int64_t cq = (c - cr) >> prm.lgN;
    const int v0 = 2 * i_pt;

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
    const int64_t R0 = m0 - cq - 1;
    const int row_bytes = N / 4 * 5;

    const int e = lane & 1;
    const uint32_t boff = (uint32_t)(5 * (lane >> 1) + e);
    const uint32_t sh = boff & 3;
    const uint32_t sel = (sh + 3) | ((sh + 2) << 4) | ((sh + 1) << 8) | (sh << 12);
    const uint32_t rd_addr = ring_s + (boff >> 2) * 4u;
    const uint32_t sha = e ? 12u : 0u;

    // batch copy: 4 rows x 2 pols x NP pieces x 5 copies of CB bytes
    const uint8_t *src[NT];
    uint32_t dst[NT];
    int trow[NT];
    const int64_t lo64 = -R0, hi64 = prm.rows_in - R0;
    const int q_lo = (int)max((int64_t)-0x3fffffff, min(lo64, (int64_t)0x3fffffff));
    const int q_hi = (int)max((int64_t)-0x3fffffff, min(hi64, (int64_t)0x3fffffff));
    const uint32_t span = (uint32_t)max(q_hi - q_lo, 0);
#pragma unroll
    for (int t = 0; t < NT; ++t) {
        const int cidx = lane + 32 * t;
        const bool has = cidx < NCH;
        const int cc = has ? cidx : 0;
        const int row = cc / (10 * NP), rem = cc - row * (10 * NP);
        const int pol = rem / (5 * NP), k = rem - pol * (5 * NP);
        const int piece = k / 5, kk = k - piece * 5;
        const int p0 = 32 * fw + piece * (32 / NP);
        const int ip = i0 + (p0 % IL) + M * (p0 / IL);      // first point of the piece: a multiple of 32 / NP
        dst[t] = ring_s + (uint32_t)(row * kFir2SlotBytes + pol * kFir2SegBytes + k * CB);
        src[t] = abase + pol * prm.stream_bytes + (R0 + row) * (int64_t)row_bytes + (ip / 2) * 5 + kk * CB;
        trow[t] = has ? row - q_lo : -0x40000000;
    }
    const int64_t batch_bytes = (int64_t)kFirBatch * row_bytes;
    auto issue_batch = [&](int slot0) {
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            if (NT * 32 == NCH || trow[t] > -0x3fffffff) {      // lanes without a copy in this round skip it
                const uint32_t ok = (uint32_t)trow[t] < span ? (uint32_t)CB : 0u;
                ring_fill_n<CB>(dst[t] + slot0 * kFir2SlotBytes, src[t], ok);
            }
            src[t] += batch_bytes;
            if (trow[t] > -0x3fffffff) trow[t] += kFirBatch;
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    __syncwarp();
#pragma unroll
    for (int b = 0; b < kFirRingBatches - 1; ++b) issue_batch(b * kFirBatch);

    f2 acc0[T], acc1[T];
#pragma unroll
    for (int j = 0; j < T; ++j) acc0[j] = acc1[j] = f2(0.f, 0.f);
    float4 prev = make_float4(0.f, 0.f, 0.f, 0.f);

    auto load_raw = [&](int slot, uint32_t (&raw)[4]) {
        const uint32_t ad = rd_addr + slot * kFir2SlotBytes;
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(raw[0]) : "r"(ad) : "memory");
        asm volatile("ld.shared.u32 %0, [%1+4];" : "=r"(raw[1]) : "r"(ad) : "memory");
        asm volatile("ld.shared.u32 %0, [%1+80];" : "=r"(raw[2]) : "r"(ad) : "memory");
        asm volatile("ld.shared.u32 %0, [%1+84];" : "=r"(raw[3]) : "r"(ad) : "memory");
    };
    uint32_t nxt[4];
    cp_async_wait<kFirRingBatches - 2>();
    __syncwarp();
    issue_batch((kFirRingBatches - 1) * kFirBatch);
    load_raw(0, nxt);

    const int n_steps = n_out + T;
    for (int i0s = 0; i0s < n_steps; i0s += U) {
#pragma unroll
        for (int ii = 0; ii < U; ++ii) {
            if (ii % 8 == 0) {
                // the tile block gx & 1 must have been read by the butterfly warps two blocks ago
                if (gx >= 2) mbar_wait(empty0 + 8 * (gx & 1u), ((gx >> 1) - 1u) & 1u);
            }
            const uint32_t P0a = nxt[0], P0b = nxt[1], P1a = nxt[2], P1b = nxt[3];
            if ((ii + 1) % kFirBatch == 0) {
                cp_async_wait<kFirRingBatches - 2>();
                __syncwarp();
                issue_batch((((ii + 1) / kFirBatch + kFirRingBatches - 1) % kFirRingBatches) * kFirBatch);
            }
            load_raw((ii + 1) % kFirDepth, nxt);
            const uint32_t be0 = __byte_perm(P0a, P0b, sel) << sha;
            const uint32_t be1 = __byte_perm(P1a, P1b, sel) << sha;
            const f2 s0((float)((int32_t)be0 >> 22), (float)((int32_t)be1 >> 22));
            const f2 s1((float)((int32_t)(be0 << 10) >> 22), (float)((int32_t)(be1 << 10) >> 22));
            acc0[ii % T] = s0 * w0[0];
#pragma unroll
            for (int j = 1; j < T; ++j) acc0[(ii + T - j) % T] = fma_(s0, w0[j], acc0[(ii + T - j) % T]);
            acc1[ii % T] = s1 * w1[0];
#pragma unroll
            for (int j = 1; j < T; ++j) acc1[(ii + T - j) % T] = fma_(s1, w1[j], acc1[(ii + T - j) % T]);
            const f2 d0 = acc0[(ii + 1) % T], d1 = acc1[(ii + 1) % T];
            const float4 now = make_float4(d0.v.x, d0.v.y, d1.v.x, d1.v.y);       // {Re p0, Re p1, Im p0, Im p1}
            float4 cur;
            cur.x = lagc[0] ? prev.x : now.x;
            cur.y = lagc[0] ? prev.y : now.y;
            cur.z = lagc[1] ? prev.z : now.z;
            cur.w = lagc[1] ? prev.w : now.w;
            prev = now;
            sts_f4(tile_thr + ii * (256 * 16), cur);
            if (ii % 8 == 7) {
                __syncwarp();
                if (lane == 0) mbar_arrive(full0 + 8 * (gx & 1u));
                ++gx;
            }
        }
    }
    cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------------------------
// producer: butterfly warps (stage 1 of the transform)
// ---------------------------------------------------------------------------------------------------------------
// K1 = 16: thread (r = bt / 16, il = bt % 16) of the 128 butterfly threads takes row r of a block and the sixteen
// points il + 16 q of the tile, and writes y[ka][i0 + il], ka < 16.  The twiddles W_n^{(i0 + il) ka} belong to the
// thread for the whole kernel (registers).
template <int T, int K1, int M>
__device__ __forceinline__ void split_bf_run(const Fir2Params &prm, int a, int i0, int bt, uint32_t tile_s, int64_t m0,
                                             int n_out, const float2 (&tw)[K1], uint32_t full0, uint32_t empty0, unsigned &gx)
{
    static_assert(K1 == 16, "stage-1 radix 16");
    constexpr int IL = 256 / K1;
    const int lane = threadIdx.x & 31;
    const int il = bt % IL, r = bt / IL;
    const int n_blocks = (n_out + T + kFirUnroll - 1) / kFirUnroll * (kFirUnroll / 8);
    for (int x = 0; x < n_blocks; ++x) {
        mbar_wait(full0 + 8 * (gx & 1u), (gx >> 1) & 1u);
        const int rho = 8 * x - T + r;                          // row of the run in this thread's tile slot
        cx<f2> v[K1];
        const bool valid = rho >= 0 && rho < n_out;
        if (valid) {
            const uint32_t s0 = tile_s + (uint32_t)((((8 * x + r) & (kSplitTileSlots - 1)) * 256 + il) * 16);
#pragma unroll
            for (int q = 0; q < K1; ++q) v[q] = unpack_unit(lds_f4(s0 + q * IL * 16));
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty0 + 8 * (gx & 1u));     // release: the loads above have completed
        ++gx;
        if (valid) {
            Dif<K1, f2>::run(v);
            float4 *yp = reinterpret_cast<float4 *>(prm.g) +
                         (((int64_t)a * prm.chunk_cap + (m0 + rho - prm.m_begin)) * K1) * M + i0 + il;
#pragma unroll
            for (int ka = 0; ka < K1; ++ka) {
                cx<f2> y = v[ka];
                if (ka > 0) y = cmul(v[ka], tw[ka].x, tw[ka].y);
                stg_stream_f4(yp + ka * M, pack_unit(y));
            }
        }
    }
}

constexpr size_t split_producer_smem() { return (size_t)kSplitTileBytes + kSplitFirWarps * kSplitRingBytes + 64; }

// grid: (n / 256 slices, row tiles, antennas); 8 FIR warps + 4 butterfly warps
#ifndef FE_SPLIT_LB
#define FE_SPLIT_LB kSplitProducerThreads
#endif
template <int T, int K1, int M = kSubM>
__global__ void __launch_bounds__(FE_SPLIT_LB, 1) split_fir_kernel(const __grid_constant__ SplitParams prm)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int IL = 256 / K1;                                 // consecutive i' per q: the CTA holds 256 points
    const int tid = threadIdx.x, warp = tid >> 5;
    const uint32_t s_base = smem_u32(smem_raw);
    const uint32_t tile_s = s_base;
    const uint32_t bar0 = s_base + kSplitTileBytes + kSplitFirWarps * kSplitRingBytes;
    const uint32_t full0 = bar0, empty0 = bar0 + 16;
    if (tid == 0) {
        mbar_init(full0, kSplitFirWarps);
        mbar_init(full0 + 8, kSplitFirWarps);
        mbar_init(empty0, kSplitBfWarps);
        mbar_init(empty0 + 8, kSplitBfWarps);
        mbar_fence_init();
    }
    __syncthreads();

    const int a = blockIdx.z;
    const int i0 = (int)blockIdx.x * IL;
    const int64_t m_first = prm.fir.m_begin + (int64_t)blockIdx.y * prm.fir.rows_per_tile;
    const int64_t m_stop = min(m_first + (int64_t)prm.fir.rows_per_tile, prm.fir.m_end);
    const int32_t *ctab = prm.fir.coarse + (int64_t)a * 2 * prm.fir.n_coarse;
    // both roles walk the same runs (maximal stretches of spectra with one coarse delay)
    auto next_run = [&](int64_t m, int32_t &c) {
        c = ctab[prm.fir.n_coarse == 1 ? 0 : m];
        int64_t run_end = m_stop;
        if (prm.fir.n_coarse != 1) {
            run_end = m + 1;
            while (run_end < m_stop && ctab[run_end] == c) ++run_end;
        }
        return run_end;
    };
    unsigned gx = 0;
    if (warp < kSplitFirWarps) {
        const uint32_t ring_s = s_base + kSplitTileBytes + warp * kSplitRingBytes;
        const uint8_t *abase = prm.fir.in + (int64_t)a * 2 * prm.fir.stream_bytes;
        for (int64_t m = m_first; m < m_stop;) {
            int32_t c;
            const int64_t run_end = next_run(m, c);
            split_fir_run<T, IL, M>(prm.fir, abase, i0, warp, ring_s, (int64_t)c, m, (int)(run_end - m), tile_s + (uint32_t)tid * 16u,
                                 full0, empty0, gx);
            m = run_end;
        }
    } else {
        const int bt = tid - 32 * kSplitFirWarps;
        float2 tw[K1];
#pragma unroll
        for (int ka = 0; ka < K1; ++ka) tw[ka] = __ldg(prm.tw1 + ka * M + i0 + bt % IL);
        for (int64_t m = m_first; m < m_stop;) {
            int32_t c;
            const int64_t run_end = next_run(m, c);
            split_bf_run<T, K1, M>(prm.fir, a, i0, bt, tile_s, m, (int)(run_end - m), tw, full0, empty0, gx);
            m = run_end;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// consumer: stage 2 of the transform and the epilogue
// ---------------------------------------------------------------------------------------------------------------
// The consumers read the gain (x rotation) table in "split order", entry (k mod K1) * M + k / K1 for channel k: the
// threads of a transform ka hold the channels ka + K1 k' with consecutive k', which natural order would spread over one
// 128-byte line per lane.
template <int K1, int M>
__device__ __forceinline__ int split_gidx(int k) { return (k & (K1 - 1)) * M + k / K1; }

static __global__ void permute_rg2_split(float4 *dst, const float4 *src, int n, int K1, int A)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int a = blockIdx.y;
    if (k >= n || a >= A) return;
    dst[(int64_t)a * n + (k % K1) * (n / K1) + k / K1] = src[(int64_t)a * n + k];
}

struct SplitPhase {          // per spectrum, per-spectrum delay mode only; units {re p0, re p1, im p0, im p1}
    float4 ea[32];           // exp(i phi) exp(-2 pi i d_eff ka / N), ka < K1
    float4 et[16];           // exp(-2 pi i d_eff K1 t / N)
    float4 step[9];          // exp(-2 pi i d_eff 16 K1 kq / N), kq <= 8
    float4 c3;               // exp(2 i phi) exp(-i pi d_eff): E[n - k] = c3 conj(E[k])
};

// warp p (< 2) of the team sets up pol p's phasors of spectrum (a, m); d_eff = d + cr, the cr part reduced exactly
template <int K1>
__device__ __forceinline__ void split_setup_phase(const Fft2Params &prm, SplitPhase *sph, int a, int64_t m, int p, int lane)
{
    constexpr int N = 2 * K1 * kSubM;
    const int64_t st = (int64_t)a * 2 + p;
    const int32_t c = prm.coarse[st * prm.n_coarse + (prm.n_coarse == 1 ? 0 : m)];
    const int cr = (int)(c & (N - 1));
    const double d = (double)prm.fine_d[st * prm.n_fine + (prm.n_fine == 1 ? 0 : m)];
    const double phi = (double)prm.fine_phi[st * prm.n_fine + (prm.n_fine == 1 ? 0 : m)];
    auto phasor = [&](int k) { return phasor_turns(-(d / (double)N) * (double)k - (double)((cr * k) & (N - 1)) / (double)N); };
    auto put = [&](float4 *dst4, float2 v) {
        float *dst = reinterpret_cast<float *>(dst4);
        dst[p] = v.x;
        dst[2 + p] = v.y;
    };
    double sphi, cphi;
    sincos(phi, &sphi, &cphi);
    const float2 ephi = make_float2((float)cphi, (float)sphi);
    if (lane < K1) put(&sph->ea[lane], cmulf(phasor(lane), ephi));
    if (lane < 16) put(&sph->et[lane], phasor(K1 * lane));
    if (lane >= 16 && lane < 25) put(&sph->step[lane - 16], phasor(16 * K1 * (lane - 16)));
    if (lane == 25) {
        double s, c_;
        sincos(2.0 * phi, &s, &c_);
        const float2 e2 = make_float2((float)c_, (float)s);
        float2 h = phasor_turns(-0.5 * d);                // exp(-i pi d_eff) = exp(-i pi d) (-1)^cr
        if (cr & 1) { h.x = -h.x; h.y = -h.y; }
        put(&sph->c3, cmulf(e2, h));
    }
}

// post-twiddle, rotation x gain, and the 4-byte word / float4 of channel kA and of its mirror kB
template <int K1, bool F32OUT>
__device__ __forceinline__ void split_epilogue(cx<f2> zk, cx<f2> zm, float2 tp, cx<f2> rgA, cx<f2> rgB, int kA, int kB,
                                               uint32_t *stage, float4 *yout)
{
    constexpr int n = K1 * kSubM;
    const f2 sr = zk.re + zm.re, si = zk.im - zm.im;      // S = Z[k] + conj Z[n-k]
    const f2 dr = zk.re - zm.re, di = zk.im + zm.im;      // D = Z[k] - conj Z[n-k]
    const f2 fr = fnma_(di, tp.y, dr * tp.x);             // F = D * (i w^k)
    const f2 fi = fma_(di, tp.x, dr * tp.y);
    const cx<f2> xk = {sr - fr, si - fi};                 // 2 X[k]
    const cx<f2> xm = {sr + fr, -(si + fi)};              // 2 X[n-k] = conj(S + F)
    const cx<f2> yA = cmul2(xk, rgA), yB = cmul2(xm, rgB);
    if (F32OUT) {
        yout[kA] = make_float4(yA.re.v.x, yA.im.v.x, yA.re.v.y, yA.im.v.y);
        if (kB < n) yout[kB] = make_float4(yB.re.v.x, yB.im.v.x, yB.re.v.y, yB.im.v.y);
    } else {
        stage[(kA % K1) * kStagePitch + kA / K1] = quantize_unit(yA);
        if (kB < n) stage[(kB % K1) * kStagePitch + kB / K1] = quantize_unit(yB);
    }
}

// One warp: the 256-point transforms ka0 = pair, ka1 = K1 - pair of spectrum (a, m) (pair 0: ka = 0 and K1 / 2, which
// mirror onto themselves).  yrow = y[.][.] of the spectrum, xb = the warp's exchange buffer (2 * kXHalf units).
template <int K1, bool F32OUT>
__device__ __forceinline__ void split_sub256_pair(const Fft2Params &prm, const float2 *__restrict__ tw256, int pair,
                                                  const float4 *__restrict__ yrow, float4 *xb, uint32_t *stage, float4 *yout,
                                                  int a, const SplitPhase *sph)
{
    constexpr int n = K1 * kSubM;
    const int lane = threadIdx.x & 31, h = lane >> 4, t = lane & 15;
    const int ka = pair == 0 ? (h ? K1 / 2 : 0) : (h ? K1 - pair : pair);
    float4 *xh = xb + h * kXHalf;

    cx<f2> x[16];
    {
        const float4 *src = yrow + ka * kSubM + t;
#pragma unroll
        for (int r = 0; r < 16; ++r) x[r] = unpack_unit(ldg_stream_f4(src + 16 * r));
    }
    Dif<16, f2>::run(x);
#pragma unroll
    for (int kb = 0; kb < 16; ++kb) {
        cx<f2> y = x[kb];
        if (kb > 0) {
            const float2 w = __ldg(tw256 + kb * 16 + t);
            y = cmul(x[kb], w.x, w.y);
        }
        xh[kb * 17 + t] = pack_unit(y);
    }
    __syncwarp();
    float4 *mine = xh + t * 17;
#pragma unroll
    for (int j = 0; j < 16; ++j) x[j] = unpack_unit(mine[j]);
    Dif<16, f2>::run(x);                                  // x[kc] = Z[ka + K1 (t + 16 kc)]

    // mirror exchange: the upper half, reversed, into this thread's own row; the partner reads it
    const bool special = pair == 0 && lane == 0;
    if (special) {
#pragma unroll
        for (int j = 0; j < 8; ++j) mine[j] = pack_unit(x[(16 - j) % 16]);
        mine[8] = pack_unit(x[8]);
    } else {
#pragma unroll
        for (int j = 0; j < 8; ++j) mine[j] = pack_unit(x[15 - j]);
    }
    const float4 *theirs;
    if (pair != 0)
        theirs = xb + (1 - h) * kXHalf + (15 - t) * 17;
    else
        theirs = xh + (h ? 15 - t : (16 - t) & 15) * 17;

    const int k0 = ka + K1 * t;
    const float2 tpK = __ldg(prm.tpost + k0);
    const float4 *__restrict__ gtab = reinterpret_cast<const float4 *>(prm.rg2) + (int64_t)a * n;
    cx<f2> base = {f2(1.f, 1.f), f2(0.f, 0.f)};
    if (prm.per_spectrum) base = cmul2(unpack_unit(sph->ea[ka]), unpack_unit(sph->et[t]));
    auto rot_gain = [&](int kq, cx<f2> gA_, cx<f2> gB_, cx<f2> &rgA, cx<f2> &rgB) {
        if (prm.per_spectrum) {
            const cx<f2> E = cmul2(base, unpack_unit(sph->step[kq]));
            const cx<f2> Ec = {E.re, -E.im};
            const cx<f2> eA = {E.re * 0.5f, E.im * 0.5f};
            const cx<f2> eB0 = cmul2(unpack_unit(sph->c3), Ec);
            const cx<f2> eB = {eB0.re * 0.5f, eB0.im * 0.5f};
            rgA = cmul2(eA, gA_);
            rgB = cmul2(eB, gB_);
        } else {
            rgA = gA_;
            rgB = gB_;
        }
    };
    float4 gA[8], gB[8];
#pragma unroll
    for (int kq = 0; kq < 8; ++kq) {
        const int kA = k0 + 16 * K1 * kq;
        gA[kq] = ldg_keep_f4(gtab + split_gidx<K1, kSubM>(kA));
        gB[kq] = ldg_keep_f4(gtab + split_gidx<K1, kSubM>((n - kA) & (n - 1)));
    }
    __syncwarp();
#pragma unroll
    for (int kq = 0; kq < 8; ++kq) {
        const int kA = k0 + 16 * K1 * kq, kB = n - kA;      // kB == n for the DC channel (dropped Nyquist)
        const cx<f2> zm = unpack_unit(theirs[kq]);
        cx<f2> rgA, rgB;
        rot_gain(kq, unpack_unit(gA[kq]), unpack_unit(gB[kq]), rgA, rgB);
        float2 tp = tpK;
        if (kq > 0) {                                     // (sin, cos)(2 pi kA / N): the thread's own word rotated by 2 pi kq / 32
            const float cphi = w32_cos(kq), sphi = w32_sin(kq);
            tp = make_float2(fmaf(tpK.x, cphi, tpK.y * sphi), fmaf(-tpK.x, sphi, tpK.y * cphi));
        }
        split_epilogue<K1, F32OUT>(x[kq], zm, tp, rgA, rgB, kA, kB, stage, yout);
    }
    if (special) {                                        // channel n/2 mirrors onto itself
        const cx<f2> zh = unpack_unit(mine[8]);
        cx<f2> rgA, rgB;
        const cx<f2> gh = unpack_unit(__ldg(gtab + split_gidx<K1, kSubM>(n / 2)));
        rot_gain(8, gh, gh, rgA, rgB);
        split_epilogue<K1, F32OUT>(zh, zh, make_float2(1.0f, 0.0f), rgA, rgB, n / 2, n, stage, yout);
    }
    __syncwarp();                                         // the exchange buffer is reused by the next pair
}

// staged int8 words of one spectrum -> global, 16 bytes per thread and step, consecutive threads consecutive bytes
template <int K1>
__device__ __forceinline__ void split_stage_out(const uint32_t *stage, uint4 *rec, int tid, int n_threads)
{
    constexpr int n = K1 * kSubM, QD = K1 / 4;
    for (int cidx = tid; cidx < n / 4; cidx += n_threads) {
        const int kp = cidx / QD, qd = cidx - kp * QD;
        const uint32_t *s = stage + (4 * qd) * kStagePitch + kp;
        stg_stream_u4(rec + cidx, make_uint4(s[0], s[kStagePitch], s[2 * kStagePitch], s[3 * kStagePitch]));
    }
}

template <int K1>
struct SplitFftSmem {
    static constexpr int warps = K1 / 2 < 8 ? K1 / 2 : 8;                  // warps of the team that shares a spectrum
    static constexpr size_t xchg_off = 0;
    static constexpr size_t stage_off = (size_t)warps * 2 * kXHalf * 16;
    static constexpr size_t phase_off = stage_off + (size_t)K1 * kStagePitch * 4;
    static constexpr size_t bytes = phase_off + sizeof(SplitPhase);
};

// one CTA per (antenna, spectrum): warp w does the pairs w, w + warps, ...
template <int K1, bool F32OUT>
__global__ void __launch_bounds__(SplitFftSmem<K1>::warps * 32, 2) split_fft_kernel(const __grid_constant__ SplitParams prm)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using SM = SplitFftSmem<K1>;
    constexpr int n = K1 * kSubM;
    const int tid = threadIdx.x, warp = tid >> 5;
    const int a = (int)gridDim.y - 1 - (int)blockIdx.y;                    // reverse of the producer's order (L2 hits)
    const int64_t m = prm.fft.m_end - 1 - (int64_t)blockIdx.x;
    if (m < prm.fft.m_begin) return;
    float4 *xb = reinterpret_cast<float4 *>(smem_raw + SM::xchg_off) + warp * 2 * kXHalf;
    uint32_t *stage = reinterpret_cast<uint32_t *>(smem_raw + SM::stage_off);
    SplitPhase *sph = reinterpret_cast<SplitPhase *>(smem_raw + SM::phase_off);
    if (prm.fft.per_spectrum) {
        if (warp < 2) split_setup_phase<K1>(prm.fft, sph, a, m, warp, tid & 31);
        __syncthreads();
    }
    const float4 *yrow = reinterpret_cast<const float4 *>(prm.fft.g) + ((int64_t)a * prm.fft.chunk_cap + (m - prm.fft.m_begin)) * n;
    float4 *yout = F32OUT ? reinterpret_cast<float4 *>(prm.fft.out_f32 + (((int64_t)a * prm.fft.n_spectra + m) * n) * 4) : nullptr;
    for (int pair = warp; pair < K1 / 2; pair += SM::warps)
        split_sub256_pair<K1, F32OUT>(prm.fft, prm.tw256, pair, yrow, xb, stage, yout, a, sph);
    if (!F32OUT) {
        __syncthreads();
        uint4 *rec = reinterpret_cast<uint4 *>(prm.fft.out + (((int64_t)a * prm.fft.n_spectra + m) * n) * 4);
        split_stage_out<K1>(stage, rec, tid, SM::warps * 32);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// consumer for n >= 16384: stage 2 is K1 = 16 transforms of M = n / 16 = 1024 or 2048 points, too large for a warp.
// One CTA = two teams of Plan::tpf threads, one team per transform of the mirror pair (ka, K1 - ka); each team runs
// passes 1 and 2 of the pol-packed M-point plan of fe_fft2.cuh in its own exchange buffer, and the last pass takes
// the mirror halves out of the OTHER team's buffer (pair 0: ka = 0 and K1 / 2 mirror onto themselves).  This replaces
// the pol-sequential four-pass transform of fe_fft.cuh, which needs two sweeps over the row at n = 32768 because the
// whole row does not fit one SM's shared memory (BASELINE.json north_star (b): "a four-step decomposition through
// HBM ... for n = 32768").  A transform ka holds the channels k = ka (mod 16), so a thread's output words are 64
// bytes apart; the eight CTAs of a spectrum run side by side and their words meet in L2.
// ---------------------------------------------------------------------------------------------------------------
struct SplitPhaseBig {       // per (CTA, spectrum), per-spectrum delay mode only; units {re p0, re p1, im p0, im p1}
    float4 ea[2];            // [team]: exp(i phi) exp(-2 pi i d_eff ka / N)
    float4 elo[16];          // exp(-2 pi i d_eff K1 K_lo / N)
    float4 ehi[16];          // exp(-2 pi i d_eff K1 16 K_hi / N)
    float4 step[9];          // exp(-2 pi i d_eff K1 Q kq / N), kq <= R3 / 2
    float4 c3;               // exp(2 i phi) exp(-i pi d_eff)
};

template <class Plan, int K1>
__device__ __forceinline__ void split_big_setup_phase(const Fft2Params &prm, SplitPhaseBig *sph, int a, int64_t m, int pair,
                                                      int p, int lane)
{
    constexpr int N = 2 * K1 * Plan::n, Q = Plan::Q, H = Plan::R3 / 2;
    const int64_t st = (int64_t)a * 2 + p;
    const int32_t c = prm.coarse[st * prm.n_coarse + (prm.n_coarse == 1 ? 0 : m)];
    const int cr = (int)(c & (N - 1));
    const double d = (double)prm.fine_d[st * prm.n_fine + (prm.n_fine == 1 ? 0 : m)];
    const double phi = (double)prm.fine_phi[st * prm.n_fine + (prm.n_fine == 1 ? 0 : m)];
    auto phasor = [&](int k) { return phasor_turns(-(d / (double)N) * (double)k - (double)(((int64_t)cr * k) & (N - 1)) / (double)N); };
    auto put = [&](float4 *dst4, float2 v) {
        float *dst = reinterpret_cast<float *>(dst4);
        dst[p] = v.x;
        dst[2 + p] = v.y;
    };
    double sphi, cphi;
    sincos(phi, &sphi, &cphi);
    const float2 ephi = make_float2((float)cphi, (float)sphi);
    if (lane < 2) put(&sph->ea[lane], cmulf(phasor(pair == 0 ? (lane ? K1 / 2 : 0) : (lane ? K1 - pair : pair)), ephi));
    if (lane < 16) put(&sph->elo[lane], phasor(K1 * lane));
    if (lane >= 16 && lane < 16 + Q / 16) put(&sph->ehi[lane - 16], phasor(K1 * 16 * (lane - 16)));
    if (lane < H + 1) put(&sph->step[lane], phasor(K1 * Q * lane));
    if (lane == 31) {
        double s, c_;
        sincos(2.0 * phi, &s, &c_);
        const float2 e2 = make_float2((float)c_, (float)s);
        float2 h = phasor_turns(-0.5 * d);
        if (cr & 1) { h.x = -h.x; h.y = -h.y; }
        put(&sph->c3, cmulf(e2, h));
    }
}

template <class Plan>
struct SplitBigSmem {
    static constexpr uint32_t buf_bytes = ((uint32_t)Plan::units * 16u + 127u) & ~127u;
    static constexpr uint32_t phase_off = 2 * buf_bytes;
    static constexpr size_t bytes = phase_off + sizeof(SplitPhaseBig);
};

// Output of the pair kernel: a transform ka holds the channels ka (mod 16), so a thread's int8 words are 64 bytes
// apart and every 4-byte store is its own L2 sector; the eight CTAs of a spectrum run side by side and their words
// meet in L2.  Collecting the words per eighth of the spectrum through a cluster's distributed shared memory
// (st.shared::cluster into the owner CTA's staging buffer, one cluster barrier, then full-line stores) was built and
// measured SLOWER (1.02 -> 1.70 ms for config 3: 4096 remote 4-byte stores per CTA at the ~20 B/clk of the SM-to-SM
// network, plus the co-scheduling of 8-CTA clusters), so the direct stores stay.
// grid (K1 / 2 pairs, spectra of the chunk, antennas); 2 * Plan::tpf threads
template <class Plan, int K1, bool F32OUT>
__global__ void __launch_bounds__(2 * Plan::tpf, 512 / (2 * Plan::tpf)) split_pair_kernel(const __grid_constant__ SplitParams sp)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using SM = SplitBigSmem<Plan>;
    constexpr int M = Plan::n, n = K1 * M, R = Plan::R3, H = R / 2, Q = Plan::Q, tpf = Plan::tpf;
    static_assert(Plan::SW == 1 && Q == tpf, "one-sweep plan, one residue per thread");
    const Fft2Params &prm = sp.fft;
    const int team = threadIdx.x / tpf, K = threadIdx.x - team * tpf;
    const int pair = blockIdx.x;
    const int a = blockIdx.z;
    const int64_t m = prm.m_begin + blockIdx.y;
    const int ka = pair == 0 ? (team ? K1 / 2 : 0) : (team ? K1 - pair : pair);
    float4 *sm = reinterpret_cast<float4 *>(smem_raw + (size_t)team * SM::buf_bytes);
    const float4 *other = reinterpret_cast<const float4 *>(smem_raw + (size_t)(pair == 0 ? team : 1 - team) * SM::buf_bytes);
    SplitPhaseBig *sph = reinterpret_cast<SplitPhaseBig *>(smem_raw + SM::phase_off);
    if (prm.per_spectrum && threadIdx.x < 64) split_big_setup_phase<Plan, K1>(prm, sph, a, m, pair, threadIdx.x >> 5, threadIdx.x & 31);

    // passes 1 and 2 of the M-point transform of y[ka][.] (pass twiddles of the M-point plan)
    const RowInGlobal yrow{reinterpret_cast<const float4 *>(prm.g) + (((int64_t)a * prm.chunk_cap + (m - prm.m_begin)) * K1 + ka) * (int64_t)M};
    fft2_pass1<Plan>(yrow, sm, sp.ptw1, K);
    __syncthreads();
    fft2_pass2<Plan>(sm, sp.ptw2, K);
    __syncthreads();

    // last pass: residue K of this transform, Z[ka + K1 (K + Q kq)]
    const bool self0 = pair == 0 && team == 0;                 // ka = 0 mirrors onto itself with the index shifted by one
    const bool special = self0 && K == 0;
    float4 *mine = sm + (K & (Plan::R1 - 1)) * Plan::blk + (K / Plan::R1) * Plan::M2;
    const int Kp = self0 ? (Q - K) & (Q - 1) : Q - 1 - K;
    const float4 *theirs = other + (Kp & (Plan::R1 - 1)) * Plan::blk + (Kp / Plan::R1) * Plan::M2;
    cx<f2> z[R];
#pragma unroll
    for (int t = 0; t < R; ++t) z[t] = unpack_unit(mine[t]);
    Dif<R, f2>::run(z);
    if (special) {
#pragma unroll
        for (int j = 0; j < H; ++j) mine[j] = pack_unit(z[(R - j) % R]);
        mine[H] = pack_unit(z[H]);
    } else {
#pragma unroll
        for (int j = 0; j < H; ++j) mine[j] = pack_unit(z[R - 1 - j]);
    }

    const int k0 = ka + K1 * K;
    const float2 tpK = __ldg(prm.tpost + k0);
    const float4 *__restrict__ gtab = reinterpret_cast<const float4 *>(prm.rg2) + (int64_t)a * n;
    float4 *yout = F32OUT ? reinterpret_cast<float4 *>(prm.out_f32 + (((int64_t)a * prm.n_spectra + m) * n) * 4) : nullptr;
    uint32_t *rec = F32OUT ? nullptr : reinterpret_cast<uint32_t *>(prm.out + (((int64_t)a * prm.n_spectra + m) * n) * 4);
    // post-twiddle, rotation x gain, quantisation and store of the pair (kA, kB)
    auto finish = [&](cx<f2> zk, cx<f2> zm, float2 tp, cx<f2> rgA, cx<f2> rgB, int kA, int kB) {
        const f2 sr = zk.re + zm.re, si = zk.im - zm.im;
        const f2 dr = zk.re - zm.re, di = zk.im + zm.im;
        const f2 fr = fnma_(di, tp.y, dr * tp.x);
        const f2 fi = fma_(di, tp.x, dr * tp.y);
        const cx<f2> xk = {sr - fr, si - fi};
        const cx<f2> xm = {sr + fr, -(si + fi)};
        const cx<f2> yA = cmul2(xk, rgA), yB = cmul2(xm, rgB);
        if constexpr (F32OUT) {
            yout[kA] = make_float4(yA.re.v.x, yA.im.v.x, yA.re.v.y, yA.im.v.y);
            if (kB < n) yout[kB] = make_float4(yB.re.v.x, yB.im.v.x, yB.re.v.y, yB.im.v.y);
        } else {
            rec[kA] = quantize_unit(yA);
            if (kB < n) rec[kB] = quantize_unit(yB);
        }
    };
    float4 gA[H], gB[H];
#pragma unroll
    for (int kq = 0; kq < H; ++kq) {
        const int kA = k0 + K1 * Q * kq;
        gA[kq] = ldg_keep_f4(gtab + split_gidx<K1, M>(kA));
        gB[kq] = ldg_keep_f4(gtab + split_gidx<K1, M>((n - kA) & (n - 1)));
    }
    __syncthreads();                                           // upper halves are in the exchange buffers
    cx<f2> base = {f2(1.f, 1.f), f2(0.f, 0.f)};
    if (prm.per_spectrum)
        base = cmul2(cmul2(unpack_unit(sph->ea[team]), unpack_unit(sph->elo[K & 15])), unpack_unit(sph->ehi[K >> 4]));
    auto rot_gain = [&](int kq, cx<f2> gA_, cx<f2> gB_, cx<f2> &rgA, cx<f2> &rgB) {
        if (prm.per_spectrum) {
            const cx<f2> E = cmul2(base, unpack_unit(sph->step[kq]));
            const cx<f2> Ec = {E.re, -E.im};
            const cx<f2> eA = {E.re * 0.5f, E.im * 0.5f};
            const cx<f2> eB0 = cmul2(unpack_unit(sph->c3), Ec);
            const cx<f2> eB = {eB0.re * 0.5f, eB0.im * 0.5f};
            rgA = cmul2(eA, gA_);
            rgB = cmul2(eB, gB_);
        } else {
            rgA = gA_;
            rgB = gB_;
        }
    };
#pragma unroll
    for (int kq = 0; kq < H; ++kq) {
        const int kA = k0 + K1 * Q * kq, kB = n - kA;
        const cx<f2> zm = unpack_unit(theirs[kq]);
        cx<f2> rgA, rgB;
        rot_gain(kq, unpack_unit(gA[kq]), unpack_unit(gB[kq]), rgA, rgB);
        float2 tp = tpK;
        if (kq > 0) {                                          // (sin, cos)(2 pi kA / N): rotate the thread's word by 2 pi kq / (2 R)
            constexpr int st = 16 / R;
            const float cphi = w32_cos(kq * st), sphi = w32_sin(kq * st);
            tp = make_float2(fmaf(tpK.x, cphi, tpK.y * sphi), fmaf(-tpK.x, sphi, tpK.y * cphi));
        }
        finish(z[kq], zm, tp, rgA, rgB, kA, kB);
    }
    if (special) {                                             // channel n/2 mirrors onto itself
        const cx<f2> zh = unpack_unit(mine[H]);
        cx<f2> rgA, rgB;
        const cx<f2> gh = unpack_unit(__ldg(gtab + split_gidx<K1, M>(n / 2)));
        rot_gain(H, gh, gh, rgA, rgB);
        finish(zh, zh, make_float2(1.0f, 0.0f), rgA, rgB, n / 2, n);
    }
}

// launchers (fe_split.cu)
cudaError_t split_launch_fir(int T, int n, const SplitParams &prm, dim3 grid, bool set_attr, cudaStream_t stream);
cudaError_t split_launch_fft(int n, bool f32out, const SplitParams &prm, dim3 grid, bool set_attr, cudaStream_t stream);
bool split_supported(int n, int T);
bool split_is_big(int n);

}  // namespace fe
