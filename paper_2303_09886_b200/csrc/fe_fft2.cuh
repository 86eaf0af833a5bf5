// fe_fft2.cuh -- steps 4-7 of the path for the pol-packed layout: N-point real-to-complex FFT of BOTH
// polarisations of an (antenna, spectrum) in one CTA, fine-delay rotation
// (PAPER.md:41), gain, quantisation and the pol-interleaved int8 store.
//
// Input: scratch rows of fe_fir2.cuh, n units {Re z p0, Re z p1, Im z p0, Im z p1}, z[i] = g'[2i] + i g'[2i+1].
// n = R1*R2*R3 with R1 = 16, decimation in frequency, natural-order input:
//   pass 1, 2   packed FP32 lanes = (pol 0, pol 1): one butterfly serves both pols and every twiddle is a
//               scalar broadcast to both lanes, so the twiddle tables are read once per spectrum, not per pol;
//   pass 3      thread K transforms residue K (Z[K + Q kq]), swaps the upper half of its outputs with the thread of
//               the mirror residue Q - K through the exchange buffer, and then owns Z[k] and Z[n-k] for half of
//               its channels: real-FFT post-twiddle, rotation, gain, quantisation and the 4-byte
//               output word {re0, im0, re1, im1} of a channel all happen in registers, packed over the pols.
// Exchange buffer (in place, one __syncthreads per pass): unit (k1, rest) lives at k1*(n/16 + 1) + rest.
// The one-unit skew per k1 block makes the 128-bit accesses of pass 3 (consecutive lanes = consecutive k1)
// bank-conflict free.
#pragma once
#include <cuda_fp16.h>

#include "fe_common.cuh"
#include "fe_fft.cuh"


namespace fe {

// SW = 2 ("two sweeps", n = 8192): the first digit has radix 32; sweep h computes the top radix-2 stage of the
// radix-32 butterfly on the fly while loading (a[j] = x[j] + x[j+16], or (x[j] - x[j+16]) W_32^j for h = 1) and then
// runs the remaining n/2-point transform exactly like the one-sweep plan, producing the channels k = h (mod 2).
// A channel and its mirror n - k have the same parity, so every sweep finishes its own channels.  The scratch row
// is read once per sweep (the second read hits L2) and the exchange buffer stays at 64 KB: two CTAs per SM.
template <int N_CH, int R2_, int R3_, int TPF, int SW_ = 1>
struct Fft2Plan {
    static constexpr int n = N_CH;
    static constexpr int SW = SW_;
    static constexpr int nh = N_CH / SW_;                 // points of one sweep's transform
    static constexpr int R1 = 16, R2 = R2_, R3 = R3_;
    static constexpr int tpf = TPF;
    static constexpr int M1 = nh / R1;                    // units per k1 block (= columns of pass 1)
    static constexpr int M2 = M1 / R2;                    // = R3
    static constexpr int Q = R1 * R2;                     // residues of the last pass
    static constexpr int blk = M1 + 1;                    // skewed block stride (units)
    static constexpr int units = R1 * blk;
    static_assert(SW_ == 1 || SW_ == 2, "one or two sweeps");
    static_assert(R1 * R2_ * R3_ * SW_ == N_CH, "radices must multiply to n");
    static_assert(M2 == R3_, "three passes");
    static_assert(R3_ == 8 || R3_ == 16, "last radix 8 or 16");
    static_assert(TPF == Q && TPF % 32 == 0 && TPF >= 64, "one residue per thread in the last pass");
};

__device__ __forceinline__ cx<f2> unpack_unit_ld(float4 v) { return {f2(v.x, v.y), f2(v.z, v.w)}; }

// Where pass 1 reads the row from: the scratch in global memory (two-kernel path, streamed past the L1) or a
// shared-memory landing buffer that a bulk copy filled (pipelined kernel, fe_pipe.cuh).  operator()(i) = unit i.
struct RowInGlobal {
    const float4 *p;
    __device__ __forceinline__ float4 operator()(int i) const { return ldg_stream_f4(p + i); }
};
// FP16 scratch (option "scratch_fp16", the paper's "FP16 for the inputs ... of the FFT, with the internal computations
// done in FP32"): units of four halves {Re z p0, Re z p1, Im z p0, Im z p1}, 8 bytes
struct RowInGlobalH16 {
    const uint2 *p;
    __device__ __forceinline__ float4 operator()(int i) const
    {
        uint2 v;
        asm volatile("ld.global.cg.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p + i));
        const float2 a = __half22float2(*reinterpret_cast<const __half2 *>(&v.x));
        const float2 b = __half22float2(*reinterpret_cast<const __half2 *>(&v.y));
        return make_float4(a.x, a.y, b.x, b.y);
    }
};
struct RowInShared {
    uint32_t s;                 // shared-space address of unit 0
    __device__ __forceinline__ float4 operator()(int i) const { return lds_f4(s + (uint32_t)i * 16u); }
};
// The row in the exchange buffer's own layout (block t of M1 units at t * blk): pass 1 then works IN PLACE, thread
// `col` reads the units (t, col) and writes the units (k, col), the same 16 addresses (persistent kernel below).
template <class Plan>
struct RowInPlace {
    uint32_t s;                 // shared-space address of the buffer
    __device__ __forceinline__ float4 operator()(int i) const
    {
        return lds_f4(s + (uint32_t)(i + i / Plan::M1 * (Plan::blk - Plan::M1)) * 16u);
    }
};
// CTA-wide barrier of the one-spectrum-per-CTA kernels; the pipelined kernel passes a named barrier over its FFT team
struct SyncCta {
    __device__ __forceinline__ void operator()() const { __syncthreads(); }
};

struct Fft2Params {
    const float *g;           // scratch rows a*chunk_cap + (m - m_begin), n units of 16 bytes
    int8_t *out;              // [A][S][n][2][2] or null
    float *out_f32;           // [A][S][n][2][2] or null
    const float2 *tw1;        // [16][M1]  W_n^{k col}   (cos, -sin)
    const float2 *tw2;        // [R2][M2]  W_M1^{k lo}
    const float2 *tpost;      // [n] (sin, cos)(2 pi k / N)  =  i * exp(-2 pi i k / N)
    const float4 *rg2;        // [A][n] {re p0, re p1, im p0, im p1}: const mode 0.5 * G * rotation; per-spectrum mode G
    const int32_t *coarse;    // [A*2][n_coarse]
    const float *fine_d;      // [A*2][n_fine]
    const float *fine_phi;    // [A*2][n_fine]
    int64_t n_coarse, n_fine;
    int64_t m_begin, m_end, chunk_cap, n_spectra;
    int per_spectrum;
};

// top radix-2 stage of the radix-32 first digit, element J of sweep HS (compile-time J so that W_32^J is a constant)
template <class Plan, int HS, int J, class Row>
__device__ __forceinline__ void fft2_sweep_half(const Row &grow, int col, cx<f2> (&a)[16])
{
    if constexpr (J < 16) {
        const cx<f2> xu = unpack_unit_ld(grow(J * Plan::M1 + col));
        const cx<f2> xv = unpack_unit_ld(grow((J + 16) * Plan::M1 + col));
        if constexpr (HS == 0)
            a[J] = cadd(xu, xv);
        else
            a[J] = mul_w<32, J, f2>(csub(xu, xv));
        fft2_sweep_half<Plan, HS, J + 1, Row>(grow, col, a);
    }
}

// pass 1 of sweep HS of a two-sweep plan: outputs k1 = 2 k'' + HS, twiddle W_n^{k1 col} as a running product
template <class Plan, int HS, class Row>
__device__ __forceinline__ void fft2_pass1_sweep(const Row &grow, float4 *sm, const float2 *__restrict__ tw, int tid)
{
    constexpr int M1 = Plan::M1;
    for (int col = tid; col < M1; col += Plan::tpf) {
        cx<f2> a[16];
        const float2 w1 = __ldg(tw + M1 + col);           // W_n^{col}
        fft2_sweep_half<Plan, HS, 0, Row>(grow, col, a);
        Dif<16, f2>::run(a);
        const float2 w2 = cmulf(w1, w1);
        float2 wk = HS ? w1 : w2;
#pragma unroll
        for (int kk = 0; kk < 16; ++kk) {
            cx<f2> y = a[kk];
            if (2 * kk + HS > 0) {
                y = cmul(a[kk], wk.x, wk.y);
                if (kk + 1 < 16) wk = cmulf(wk, w2);
            }
            sm[kk * Plan::blk + col] = make_float4(y.re.v.x, y.re.v.y, y.im.v.x, y.im.v.y);
        }
    }
}

template <class Plan, class Row>
__device__ __forceinline__ void fft2_pass1(const Row &grow, float4 *sm, const float2 *__restrict__ tw, int tid)
{
    constexpr int R = Plan::R1, M1 = Plan::M1;
    for (int col = tid; col < M1; col += Plan::tpf) {
        cx<f2> x[R];
#pragma unroll
        for (int t = 0; t < R; ++t) {
            const float4 v = grow(t * M1 + col);
            x[t].re = f2(v.x, v.y);
            x[t].im = f2(v.z, v.w);
        }
        Dif<R, f2>::run(x);
        // W_n^{k col}, k = 1..15, as powers of the one table word W_n^{col} (product tree of depth <= 4: the
        // rounding error stays below 5e-7, far inside the 1e-4 budget), so pass 1 reads 8 bytes of table per
        // butterfly instead of 120 and the table never competes with the gain table for the L1
        float2 w[R];
        w[1] = __ldg(tw + M1 + col);
#pragma unroll
        for (int k = 2; k < R; ++k) w[k] = cmulf(w[k / 2], w[k - k / 2]);
#pragma unroll
        for (int k = 0; k < R; ++k) {
            cx<f2> y = x[k];
            if (k > 0) {
                y = cmul(x[k], w[k].x, w[k].y);
            }
            sm[k * Plan::blk + col] = make_float4(y.re.v.x, y.re.v.y, y.im.v.x, y.im.v.y);
        }
    }
}

template <class Plan>
__device__ __forceinline__ void fft2_pass2(float4 *sm, const float2 *__restrict__ tw, int tid)
{
    constexpr int R = Plan::R2, M2 = Plan::M2;
    for (int b = tid; b < Plan::nh / R; b += Plan::tpf) {
        const int k1 = b / M2, lo = b - k1 * M2;
        float4 *col = sm + k1 * Plan::blk + lo;
        cx<f2> x[R];
#pragma unroll
        for (int t = 0; t < R; ++t) {
            const float4 v = col[t * M2];
            x[t].re = f2(v.x, v.y);
            x[t].im = f2(v.z, v.w);
        }
        Dif<R, f2>::run(x);
#pragma unroll
        for (int k = 0; k < R; ++k) {
            cx<f2> y = x[k];
            if (k > 0) {
                const float2 w = __ldg(tw + k * M2 + lo);
                y = cmul(x[k], w.x, w.y);
            }
            col[k * M2] = make_float4(y.re.v.x, y.re.v.y, y.im.v.x, y.im.v.y);
        }
    }
}

struct SpectrumPhase2 {      // shared, filled once per spectrum in per-spectrum mode; packed {re p0, re p1, im p0, im p1}
    float4 step[16];         // exp(-2 pi i d_eff Q kq / N)
    float4 c3;               // exp(2 i phi) exp(-i pi d_eff): E[n-k] = c3 * conj(E[k]) with E incl. exp(i phi)
    float4 ephi;             // exp(i phi)
    // E(k0) of a thread's first channel k0 = h + SW (K_lo + 16 K_hi) as a product of two table words, so that the
    // double-precision sincos runs 80 times per spectrum (here) instead of twice per thread and sweep
    float4 lo[2][16];        // [sweep h][K_lo]: exp(i phi) exp(-2 pi i d_eff (h + SW K_lo) / N)
    float4 hi[16];           // [K_hi]: exp(-2 pi i d_eff 16 SW K_hi / N)
};

__device__ __forceinline__ cx<f2> unpack_unit(float4 v) { return {f2(v.x, v.y), f2(v.z, v.w)}; }
__device__ __forceinline__ float4 pack_unit(cx<f2> z) { return make_float4(z.re.v.x, z.re.v.y, z.im.v.x, z.im.v.y); }
// packed complex product (both lanes independent)
__device__ __forceinline__ cx<f2> cmul2(cx<f2> a, cx<f2> b)
{
    return {fnma_(a.im, b.im, a.re * b.re), fma_(a.im, b.re, a.re * b.im)};
}

// {re p0, im p0, re p1, im p1} int8 word: round-half-even + clamp to [-127, 127]
__device__ __forceinline__ uint32_t quantize_unit(cx<f2> y)
{
    const float magic = 12582912.0f;                      // 1.5 * 2^23: the FP32 add rounds to nearest-even
    const f2 r = f2(fminf(fmaxf(y.re.v.x, -127.0f), 127.0f), fminf(fmaxf(y.re.v.y, -127.0f), 127.0f)) + f2(magic);
    const f2 i = f2(fminf(fmaxf(y.im.v.x, -127.0f), 127.0f), fminf(fmaxf(y.im.v.y, -127.0f), 127.0f)) + f2(magic);
    const uint32_t lo = __byte_perm(__float_as_uint(r.v.x), __float_as_uint(i.v.x), 0x0040);
    const uint32_t hi = __byte_perm(__float_as_uint(r.v.y), __float_as_uint(i.v.y), 0x0040);
    return __byte_perm(lo, hi, 0x5410);
}

// Post-twiddle, rotation, gain and store of channel kA = K + Q kq and of its mirror n - kA,
// both pols in the packed lanes.  zk = Z[kA], zm = Z[n - kA]; tp = i w^kA; rgA / rgB = 0.5 * gain * rotation.
template <bool F32OUT>
__device__ __forceinline__ void fft2_epilogue(cx<f2> zk, cx<f2> zm, float2 tp, cx<f2> rgA, cx<f2> rgB, int kA, int kB,
                                              int n, uint32_t *rec, float4 *yout)
{
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
        rec[kA] = quantize_unit(yA);
        if (kB < n) rec[kB] = quantize_unit(yB);
    }
}

// Pass 3: thread K transforms residue K (packed radix-R3 butterfly, Z[K + Q kq]), hands the upper half of its
// outputs to the thread of the mirror residue Q - K through the exchange buffer (in place, its own slots), and
// finishes the channels K + Q kq, kq < R3/2, together with their mirrors n - k, whose Z values are exactly the
// upper half of residue Q - K.  Residue 0 mirrors onto itself with the index shifted by one (n - Q kq = Q (R3 - kq))
// and also owns the self-mirrored channel n/2.
// Two-sweep plans (HS = sweep): residue K of sweep HS holds the channels k = HS + SW (K + Q kq); in the odd sweep
// the mirror of residue K is residue Q - 1 - K and no residue mirrors onto itself.
template <class Plan, bool F32OUT, int HS, class Sync>
__device__ __forceinline__ void fft2_pass3(float4 *sm, const Fft2Params &prm, int a, int64_t m, int tid,
                                           const SpectrumPhase2 *sph, const Sync &sync)
{
    constexpr int R = Plan::R3, H = R / 2, Q = Plan::Q, n = Plan::n, N = 2 * n, SW = Plan::SW;
    static_assert(Plan::tpf == Q, "one residue per thread");
    const int K = tid;
    const int k0 = HS + SW * K;                           // this thread's first channel
    const bool special = HS == 0 && K == 0;
    float4 *mine = sm + (K & (Plan::R1 - 1)) * Plan::blk + (K / Plan::R1) * Plan::M2;
    const int Kp = HS ? Q - 1 - K : (Q - K) & (Q - 1);
    const float4 *theirs = sm + (Kp & (Plan::R1 - 1)) * Plan::blk + (Kp / Plan::R1) * Plan::M2;

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

    // per-thread rotation base of the per-spectrum mode: E_p(K) = exp(i phi_p) exp(-2 pi i (d_p + cr) K / N)
    cx<f2> base = {f2(1.f, 1.f), f2(0.f, 0.f)};
    const float4 *__restrict__ gtab = reinterpret_cast<const float4 *>(prm.rg2) + (int64_t)a * n;
    if (prm.per_spectrum) base = cmul2(unpack_unit(sph->lo[HS][K & 15]), unpack_unit(sph->hi[K >> 4]));
    // post-twiddle phasors without a table walk: (sin, cos)(2 pi (K + Q kq) / N) = the thread's own (sin, cos)(2 pi K / N)
    // rotated by the compile-time angle 2 pi kq Q / N (Q / N is 1/32 or 1/16), one table word per thread and spectrum
    const float2 tpK = __ldg(prm.tpost + k0);
    auto tp_of = [&](int kq) {
        constexpr int st = 32 * SW * Q / N;
        const float cphi = w32_cos(kq * st), sphi = w32_sin(kq * st);
        return make_float2(fmaf(tpK.x, cphi, tpK.y * sphi), fmaf(-tpK.x, sphi, tpK.y * cphi));
    };
    uint32_t *rec = F32OUT ? nullptr : reinterpret_cast<uint32_t *>(prm.out + (((int64_t)a * prm.n_spectra + m) * n) * 4);
    float4 *yout = F32OUT ? reinterpret_cast<float4 *>(prm.out_f32 + (((int64_t)a * prm.n_spectra + m) * n) * 4) : nullptr;

    // every gain word of this thread's channels is requested before the exchange barrier so that the L2 latency of
    // the table overlaps the barrier and the mirror loads instead of being paid once per channel pair
    float4 gA[H], gB[H];
#pragma unroll
    for (int kq = 0; kq < H; ++kq) {
        const int kA = k0 + SW * Q * kq;
        gA[kq] = ldg_keep_f4(gtab + kA);
        gB[kq] = ldg_keep_f4(gtab + ((n - kA) & (n - 1)));
    }
    auto rot_gain = [&](int kq, cx<f2> gA_, cx<f2> gB_, cx<f2> &rgA, cx<f2> &rgB) {
        if (prm.per_spectrum) {
            const cx<f2> E = cmul2(base, unpack_unit(sph->step[kq]));
            const cx<f2> Ec = {E.re, -E.im};
            const cx<f2> eA = {E.re * 0.5f, E.im * 0.5f};
            const cx<f2> c3 = unpack_unit(sph->c3);
            const cx<f2> eB0 = cmul2(c3, Ec);
            const cx<f2> eB = {eB0.re * 0.5f, eB0.im * 0.5f};
            rgA = cmul2(eA, gA_);
            rgB = cmul2(eB, gB_);
        } else {
            rgA = gA_;
            rgB = gB_;
        }
    };

    sync();                                               // upper halves are in the exchange buffer
#pragma unroll
    for (int kq = 0; kq < H; ++kq) {
        const int kA = k0 + SW * Q * kq, kB = n - kA;      // kB == n for the DC channel (dropped Nyquist)
        const cx<f2> zmk = unpack_unit(theirs[kq]);
        cx<f2> rgA, rgB;
        rot_gain(kq, unpack_unit(gA[kq]), unpack_unit(gB[kq]), rgA, rgB);
        fft2_epilogue<F32OUT>(z[kq], zmk, kq == 0 ? tpK : tp_of(kq), rgA, rgB, kA, kB, n, rec, yout);
    }
    if (special) {                                        // channel n/2 = SW * Q * H mirrors onto itself
        const cx<f2> zh = unpack_unit(mine[H]);
        cx<f2> rgA, rgB;
        const cx<f2> gh = unpack_unit(__ldg(gtab + n / 2));
        rot_gain(H, gh, gh, rgA, rgB);
        fft2_epilogue<F32OUT>(zh, zh, make_float2(1.0f, 0.0f), rgA, rgB, n / 2, n, n, rec, yout);
    }
}

// Per-spectrum phasor setup (per-spectrum mode only): warp p sets up pol p's phasors in shared memory.
template <class Plan>
__device__ __forceinline__ void fft2_setup_phase(const Fft2Params &prm, SpectrumPhase2 *sph, int a, int64_t m, int tid)
{
    constexpr int N = 2 * Plan::n;
    const int p = tid >> 5, t = tid & 31;
    if (p < 2) {                                          // warp p sets up pol p: every lane a few phasors in double
        const int64_t st = (int64_t)a * 2 + p;
        const int32_t c = prm.coarse[st * prm.n_coarse + (prm.n_coarse == 1 ? 0 : m)];
        const int cr = (int)(c & (N - 1));
        const double d = (double)prm.fine_d[st * prm.n_fine + (prm.n_fine == 1 ? 0 : m)];
        const double phi = (double)prm.fine_phi[st * prm.n_fine + (prm.n_fine == 1 ? 0 : m)];
        auto phasor = [&](int k) {                        // exp(-2 pi i (d + cr) k / N), the cr part reduced exactly
            return phasor_turns(-(d / (double)N) * (double)k - (double)((cr * k) & (N - 1)) / (double)N);
        };
        auto put = [&](float4 *dst4, float2 v) {
            float *dst = reinterpret_cast<float *>(dst4);
            dst[p] = v.x;
            dst[2 + p] = v.y;
        };
        double sphi, cphi;
        sincos(phi, &sphi, &cphi);
        const float2 ephi = make_float2((float)cphi, (float)sphi);
        if (t < 16) {
            put(&sph->step[t], phasor(Plan::SW * Plan::Q * t));
            put(&sph->lo[0][t], cmulf(phasor(Plan::SW * t), ephi));
        } else {
            const int j = t - 16;
            put(&sph->hi[j], phasor(16 * Plan::SW * j));
            put(&sph->lo[1][j], cmulf(phasor(1 + Plan::SW * j), ephi));
        }
        if (t == 16) {
            put(&sph->ephi, ephi);
            double s, c_;
            sincos(2.0 * phi, &s, &c_);
            const float2 e2 = make_float2((float)c_, (float)s);
            float2 h = phasor_turns(-0.5 * d);            // exp(-i pi d_eff) = exp(-i pi d) * (-1)^cr
            if (cr & 1) { h.x = -h.x; h.y = -h.y; }
            put(&sph->c3, cmulf(e2, h));
        }
    }
}

// One spectrum of one antenna, both pols, by the tpf threads that share `sync` (the whole CTA, or the FFT team of
// the pipelined kernel).  `after_load()` runs (on every thread) once the row has been consumed (after the barrier
// that ends the last pass 1): the pipelined kernel hands its landing buffer back to the loader there.
template <class Plan, bool F32OUT, class Row, class Sync, class AfterLoad>
__device__ __forceinline__ void fft2_row_at(const Fft2Params &prm, const Row &grow, float4 *sm, SpectrumPhase2 *sph, int a,
                                            int64_t m, int tid, const Sync &sync, AfterLoad after_load)
{
    if (prm.per_spectrum) fft2_setup_phase<Plan>(prm, sph, a, m, tid);
    if constexpr (Plan::SW == 1) {
        fft2_pass1<Plan>(grow, sm, prm.tw1, tid);
        sync();
        after_load();
        fft2_pass2<Plan>(sm, prm.tw2, tid);
        sync();
        fft2_pass3<Plan, F32OUT, 0>(sm, prm, a, m, tid, sph, sync);
    } else {
        fft2_pass1_sweep<Plan, 0>(grow, sm, prm.tw1, tid);
        sync();
        fft2_pass2<Plan>(sm, prm.tw2, tid);
        sync();
        fft2_pass3<Plan, F32OUT, 0>(sm, prm, a, m, tid, sph, sync);
        sync();                                           // the exchange buffer is reused by the odd sweep
        fft2_pass1_sweep<Plan, 1>(grow, sm, prm.tw1, tid);
        sync();
        after_load();
        fft2_pass2<Plan>(sm, prm.tw2, tid);
        sync();
        fft2_pass3<Plan, F32OUT, 1>(sm, prm, a, m, tid, sph, sync);
    }
}

template <class Plan, bool F32OUT, class Row, class Sync, class AfterLoad>
__device__ __forceinline__ void fft2_row(const Fft2Params &prm, const Row &grow, unsigned char *smem_raw, int a,
                                         int64_t m, int tid, const Sync &sync, AfterLoad after_load)
{
    fft2_row_at<Plan, F32OUT>(prm, grow, reinterpret_cast<float4 *>(smem_raw),
                              reinterpret_cast<SpectrumPhase2 *>(smem_raw + (size_t)Plan::units * 16), a, m, tid, sync, after_load);
}

template <class Plan>
constexpr size_t fft2_smem_bytes()
{
    return (size_t)Plan::units * 16 + sizeof(SpectrumPhase2);
}

// One CTA per (antenna, spectrum), both pols.
template <class Plan, bool F32OUT, bool H16 = false>
static __global__ void __launch_bounds__(Plan::tpf, (512 / Plan::tpf) > 0 ? (512 / Plan::tpf) : 1) fft2_kernel(const Fft2Params prm)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int N = 2 * Plan::n;
    // CTAs are issued in the reverse of the order in which the FIR kernel wrote the scratch (last antenna, last rows
    // first): the most recently written ~100 MB are still in L2 when this kernel starts
    const int a = (int)gridDim.y - 1 - (int)blockIdx.y;
    const int64_t m = prm.m_end - 1 - (int64_t)blockIdx.x;
    if (m < prm.m_begin) return;
    if constexpr (H16) {
        const RowInGlobalH16 grow{reinterpret_cast<const uint2 *>(prm.g + ((int64_t)a * prm.chunk_cap + (m - prm.m_begin)) * (int64_t)N)};
        fft2_row<Plan, F32OUT>(prm, grow, smem_raw, a, m, threadIdx.x, SyncCta{}, [] {});
    } else {
        const RowInGlobal grow{reinterpret_cast<const float4 *>(prm.g + ((int64_t)a * prm.chunk_cap + (m - prm.m_begin)) * (int64_t)N * 2)};
        fft2_row<Plan, F32OUT>(prm, grow, smem_raw, a, m, threadIdx.x, SyncCta{}, [] {});
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Persistent variant (one-sweep plans, n <= 4096): one CTA per SM, NT teams of Plan::tpf threads, NT + 1 exchange
// buffers.  fft2_kernel is latency bound: a CTA waits for the sixteen dependent global loads of pass 1 before it has
// anything to compute, and only one other CTA of the SM can fill the gap.  Here the rows arrive by bulk copy
// (cp.async.bulk, the "recent CUDA asynchronous APIs" of PAPER.md:213) straight into the exchange buffer's own
// skewed layout, so pass 1 runs in place out of shared memory, and they arrive EARLY: the CTA's j-th row lives in
// buffer j mod (NT + 1) and is transformed by team j mod NT; the team that finishes row j hands the buffer to the
// copy of row j + NT + 1, which lands while every team is busy with the rows in between.  Teams synchronise among
// themselves with named barriers and with the copies through one mbarrier per buffer; there is no CTA-wide barrier
// after the start.  A buffer's rows are handed from team to team (row j + NT + 1 belongs to another team than row
// j), so a team that runs ahead could meet the buffer's mbarrier two phases early, where a parity wait cannot tell
// "not yet issued" from "already landed"; the issuing thread therefore also publishes the fill count of the buffer
// in shared memory and a team waits for "fill k issued" before it waits for the phase k of the mbarrier.
template <class Plan>
struct Fft2pSmem {
    static constexpr int NT = 512 / Plan::tpf;                            // teams per CTA
    static constexpr int NB = NT + 1;                                     // buffers
    static constexpr uint32_t buf_bytes = ((uint32_t)Plan::units * 16u + 127u) & ~127u;
    static constexpr uint32_t sph_off = NB * buf_bytes;
    static constexpr uint32_t bar_off = sph_off + NT * (((uint32_t)sizeof(SpectrumPhase2) + 15u) & ~15u);
    static constexpr uint32_t gen_off = bar_off + 8 * NB;                 // int per buffer: fills issued so far - 1
    static constexpr size_t bytes = gen_off + 4 * NB;
};

template <class Plan, bool F32OUT>
static __global__ void __launch_bounds__(512, 1) fft2p_kernel(const __grid_constant__ Fft2Params prm, int A)
{
    static_assert(Plan::SW == 1, "in-place landing needs a one-sweep plan");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    using SM = Fft2pSmem<Plan>;
    constexpr int NT = SM::NT, NB = SM::NB, tpf = Plan::tpf, N = 2 * Plan::n;
    constexpr uint32_t blk_bytes = (uint32_t)Plan::M1 * 16u;              // one block of M1 units of the row
    const int team = threadIdx.x / tpf, tid = threadIdx.x - team * tpf;
    const uint32_t s_base = smem_u32(smem_raw), bar0 = s_base + SM::bar_off;
    const int len = (int)(prm.m_end - prm.m_begin), total = len * A;       // the host keeps A * len below 2^31
    const int c = blockIdx.x, G = gridDim.x;

    // row q of the call, in the reverse of the FIR kernel's write order (the newest scratch rows are still in L2)
    auto row_ptr = [&](int q, int &a, int64_t &m) {
        const int ar = q / len, x = q - ar * len;
        a = A - 1 - (int)ar;
        m = prm.m_end - 1 - x;
        return reinterpret_cast<const unsigned char *>(prm.g + ((int64_t)a * prm.chunk_cap + (m - prm.m_begin)) * (int64_t)N * 2);
    };
    auto issue = [&](int j) {                                         // one thread: row j of this CTA -> buffer j % NB
        const int q = c + j * G;
        if (q >= total) return;
        int a;
        int64_t m;
        const unsigned char *src = row_ptr(q, a, m);
        const int b = j % NB;
        const uint32_t dst = s_base + (uint32_t)b * SM::buf_bytes, bar = bar0 + 8u * b;
        fence_proxy_async();                                              // the team's shared-memory accesses before the copy's
        mbar_arrive_expect_tx(bar, (uint32_t)Plan::R1 * blk_bytes);
#pragma unroll 1
        for (int t = 0; t < Plan::R1; ++t) bulk_g2s(dst + (uint32_t)t * (uint32_t)Plan::blk * 16u, src + (size_t)t * blk_bytes, blk_bytes, bar);
        __threadfence_block();                                            // the mbarrier is armed before the fill count says so
        asm volatile("st.volatile.shared.s32 [%0], %1;" ::"r"(s_base + SM::gen_off + 4u * b), "r"(j / NB) : "memory");
    };

    if (threadIdx.x == 0) {
        for (int b = 0; b < NB; ++b) {
            mbar_init(bar0 + 8u * b, 1);
            asm volatile("st.volatile.shared.s32 [%0], %1;" ::"r"(s_base + SM::gen_off + 4u * b), "r"(-1) : "memory");
        }
        mbar_fence_init();
    }
    __syncthreads();
    if (threadIdx.x == 0)
        for (int j = 0; j < NB; ++j) issue(j);

    SpectrumPhase2 *sph = reinterpret_cast<SpectrumPhase2 *>(smem_raw + SM::sph_off + team * (((uint32_t)sizeof(SpectrumPhase2) + 15u) & ~15u));
    const auto sync = [team] { bar_sync(1 + team, tpf); };
    for (int j = team; c + j * G < total; j += NT) {
        int a;
        int64_t m;
        row_ptr(c + j * G, a, m);
        const int b = j % NB;
        for (;;) {                                                        // fill j / NB of this buffer has been issued ...
            int gen;
            asm volatile("ld.volatile.shared.s32 %0, [%1];" : "=r"(gen) : "r"(s_base + SM::gen_off + 4u * b) : "memory");
            if (gen >= j / NB) break;
            __nanosleep(40);
        }
        __threadfence_block();
        mbar_wait(bar0 + 8u * b, (uint32_t)((j / NB) & 1));              // ... and has landed
        float4 *sm = reinterpret_cast<float4 *>(smem_raw + (size_t)b * SM::buf_bytes);
        const RowInPlace<Plan> row{s_base + (uint32_t)b * SM::buf_bytes};
        fft2_row_at<Plan, F32OUT>(prm, row, sm, sph, a, m, tid, sync, [] {});
        sync();                                                           // every thread of the team is done with the buffer
        if (tid == 0) issue(j + NB);
    }
}

// Pol-interleaved table of the pol-packed epilogue, [A][n] units {re p0, re p1, im p0, im p1}:
//   const mode          0.5 * G * exp(i(-2 pi (d + cr) k / N + phi))   (rotation folded in)
//   per-spectrum mode   G                                              (rotation computed per spectrum in the kernel)
static __global__ void build_rg2_table(float4 *rg2, const float2 *gains, const int32_t *coarse, const float *fine_d,
                                const float *fine_phi, int n, int A, int per_spectrum)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int a = blockIdx.y;
    if (k >= n || a >= A) return;
    const int N = 2 * n;
    float re[2], im[2];
    for (int p = 0; p < 2; ++p) {
        const int st = a * 2 + p;
        const float2 g = gains[(int64_t)st * n + k];
        if (per_spectrum) {
            re[p] = g.x;
            im[p] = g.y;
        } else {
            const int cr = (int)(coarse[st] & (N - 1));
            const double d = (double)fine_d[st], phi = (double)fine_phi[st];
            const double turns = -d * (double)k / (double)N - (double)(((int64_t)cr * k) & (N - 1)) / (double)N;
            double s, c, sp, cp;
            sincospi(2.0 * turns, &s, &c);
            sincos(phi, &sp, &cp);
            const double rr = c * cp - s * sp, ri = c * sp + s * cp;
            re[p] = (float)(0.5 * ((double)g.x * rr - (double)g.y * ri));
            im[p] = (float)(0.5 * ((double)g.x * ri + (double)g.y * rr));
        }
    }
    rg2[(int64_t)a * n + k] = make_float4(re[0], re[1], im[0], im[1]);
}

// scalar twiddle table of one pass: tw[k][x] = W_M^{k x} = (cos, -sin)(2 pi k x / M)
static __global__ void build_scalar_twiddles(float2 *tw, int R, int S, int M)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= R * S) return;
    const int k = idx / S, x = idx - k * S;
    double s, c;
    sincospi(-2.0 * (double)((k * x) % M) / (double)M, &s, &c);
    tw[idx] = make_float2((float)c, (float)s);
}

// debug: natural-order FIR output g [A][2][S][N] from pol-packed scratch rows (a*cap + m), undoing the rotation
static __global__ void unrotate2_kernel(const float *gp, float *g_out, const int32_t *coarse, int64_t n_coarse,
                                 int64_t n_spectra, int64_t cap, int N, int A)
{
    const int64_t total = (int64_t)A * 2 * n_spectra * N;
    for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total;
         idx += (int64_t)gridDim.x * blockDim.x) {
        const int t = (int)(idx % N);
        const int64_t m = (idx / N) % n_spectra;
        const int64_t st = idx / N / n_spectra;
        const int a = (int)(st / 2), pol = (int)(st % 2);
        const int64_t c = coarse[st * n_coarse + (n_coarse == 1 ? 0 : m)];
        const int cr = (int)(c & (int64_t)(N - 1));
        const int v = (t - cr) & (N - 1);
        g_out[idx] = gp[((int64_t)a * cap + m) * N * 2 + (int64_t)(v >> 1) * 4 + (v & 1) * 2 + pol];
    }
}

}  // namespace fe
