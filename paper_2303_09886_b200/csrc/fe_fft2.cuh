// fe_fft2.cuh -- steps 4-7 of the path for the pol-packed layout: N-point real-to-complex FFT of BOTH
// polarisations of an (antenna, spectrum) in one CTA, fine-delay rotation
// (PAPER.md:41), gain, quantisation and the pol-interleaved int8 store.
//
// Input: scratch rows of fe_fir2.cuh, n units {Re z p0, Re z p1, Im z p0, Im z p1}, z[i] = g'[2i] + i g'[2i+1].
// n = R1*R2*R3 with R1 = 16, decimation in frequency, natural-order input:
//   pass 1, 2   packed FP32 lanes = (pol 0, pol 1): one butterfly serves both pols and every twiddle is a
//               scalar broadcast to both lanes, so the twiddle tables are read once per spectrum, not per pol;
//   pass 3      scalar, thread = (residue pair K / Q-K, pol): it owns Z[k] and Z[n-k] of its pol and does the
//               real-FFT post-twiddle (the paper's kernel also ran "two such FFTs ... by the
//               same thread"), the rotation, the gain and the quantisation in registers; the two
//               pols of a channel sit in neighbouring lanes and are joined by one shuffle into the 4-byte
//               output word {re0, im0, re1, im1}.
// Exchange buffer (in place, one __syncthreads per pass): unit (k1, rest) lives at k1*(n/16 + 1) + rest.
// The one-unit skew per k1 block makes the scalar 64-bit reads of pass 3 (16 lanes = 16 consecutive k1)
// bank-conflict free; pass 2 writes each unit as {re0, im0, re1, im1} so that pass 3 reads (re, im) of its
// pol with one 64-bit load.
#pragma once
#include "fe_common.cuh"
#include "fe_fft.cuh"

namespace fe {

template <int N_CH, int R2_, int R3_, int TPF>
struct Fft2Plan {
    static constexpr int n = N_CH;
    static constexpr int R1 = 16, R2 = R2_, R3 = R3_;
    static constexpr int tpf = TPF;
    static constexpr int M1 = N_CH / R1;                  // units per k1 block
    static constexpr int M2 = M1 / R2;                    // = R3
    static constexpr int Q = R1 * R2;                     // residues of the last pass
    static constexpr int blk = M1 + 1;                    // skewed block stride (units)
    static constexpr int units = R1 * blk;
    static_assert(R1 * R2_ * R3_ == N_CH, "radices must multiply to n");
    static_assert(M2 == R3_, "three passes");
    static_assert(R3_ == 8 || R3_ == 16, "last radix 8 or 16");
    static_assert(Q % 32 == 0 && TPF % 32 == 0 && TPF >= 64, "whole warps in the last pass");
};

struct Fft2Params {
    const float *g;           // scratch rows a*chunk_cap + (m - m_begin), n units of 16 bytes
    int8_t *out;              // [A][S][n][2][2] or null
    float *out_f32;           // [A][S][n][2][2] or null
    const float2 *tw1;        // [16][M1]  W_n^{k col}   (cos, -sin)
    const float2 *tw2;        // [R2][M2]  W_M1^{k lo}
    const float2 *tpost;      // [n] (sin, cos)(2 pi k / N)  =  i * exp(-2 pi i k / N)
    const float2 *rg;         // const mode: [A][2][n]  0.5 * G * exp(i(-2 pi (d + cr) k/N + phi))
    const float2 *gains;      // per-spectrum mode: [A][2][n]
    const int32_t *coarse;    // [A*2][n_coarse]
    const float *fine_d;      // [A*2][n_fine]
    const float *fine_phi;    // [A*2][n_fine]
    int64_t n_coarse, n_fine;
    int64_t m_begin, m_end, chunk_cap, n_spectra;
    int per_spectrum;
};

template <class Plan>
__device__ __forceinline__ void fft2_pass1(const float4 *__restrict__ grow, float4 *sm, const float2 *__restrict__ tw, int tid)
{
    constexpr int R = Plan::R1, M1 = Plan::M1;
    for (int col = tid; col < M1; col += Plan::tpf) {
        cx<f2> x[R];
#pragma unroll
        for (int t = 0; t < R; ++t) {
            const float4 v = ldg_stream_f4(grow + t * M1 + col);
            x[t].re = f2(v.x, v.y);
            x[t].im = f2(v.z, v.w);
        }
        Dif<R, f2>::run(x);
#pragma unroll
        for (int k = 0; k < R; ++k) {
            cx<f2> y = x[k];
            if (k > 0) {
                const float2 w = __ldg(tw + k * M1 + col);
                y = cmul(x[k], w.x, w.y);
            }
            sm[k * Plan::blk + col] = make_float4(y.re.v.x, y.re.v.y, y.im.v.x, y.im.v.y);
        }
    }
}

template <class Plan>
__device__ __forceinline__ void fft2_pass2(float4 *sm, const float2 *__restrict__ tw, int tid)
{
    constexpr int R = Plan::R2, M2 = Plan::M2;
    for (int b = tid; b < Plan::n / R; b += Plan::tpf) {
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
            col[k * M2] = make_float4(y.re.v.x, y.im.v.x, y.re.v.y, y.im.v.y);     // {re0, im0, re1, im1}
        }
    }
}

// residue K of pol p -> Z[K + Q kq], kq = 0..R3-1 (scalar butterfly)
template <class Plan>
__device__ __forceinline__ void fft2_load_residue(const float4 *sm, int K, int p, cx<float> (&z)[Plan::R3])
{
    const int k1 = K & (Plan::R1 - 1), k2 = K / Plan::R1;
    const float2 *src = reinterpret_cast<const float2 *>(sm + k1 * Plan::blk + k2 * Plan::M2) + p;
#pragma unroll
    for (int t = 0; t < Plan::R3; ++t) {
        const float2 v = src[2 * t];
        z[t] = {v.x, v.y};
    }
    Dif<Plan::R3, float>::run(z);
}

template <class Plan, bool F32OUT>
__device__ __forceinline__ void fft2_pass3(const float4 *sm, const Fft2Params &prm, int a, int64_t m, int tid,
                                           const SpectrumPhase *sph_all, const double (&dts_p)[2], const int (&cr_p)[2])
{
    constexpr int Rq = Plan::R3, Q = Plan::Q, n = Plan::n, N = 2 * n;
    const float2 *__restrict__ tpost = prm.tpost;
    for (int it = tid; it < Q; it += Plan::tpf) {
        const int p = it & 1, pidx = it >> 1;
        const int64_t st = (int64_t)a * 2 + p;
        const float2 *__restrict__ gtab = (prm.per_spectrum ? prm.gains : prm.rg) + st * n;
        const SpectrumPhase *sph = sph_all + p;
        const double d_eff_turn_scale = dts_p[p];
        const int cr = cr_p[p];
        cx<float> zA[Rq], zB[Rq];
        const bool special = pidx == 0;
        fft2_load_residue<Plan>(sm, pidx, p, zA);
        fft2_load_residue<Plan>(sm, special ? Q / 2 : Q - pidx, p, zB);

        cx<float> zhalf = zA[Rq / 2];                     // only meaningful for the special thread
        if (special) {                                    // residues 0 and Q/2 mirror onto themselves: re-pair
            cx<float> a_[Rq], b_[Rq];
#pragma unroll
            for (int i = 0; i < Rq; ++i) { a_[i] = zA[i]; b_[i] = zB[i]; }
#pragma unroll
            for (int i = 0; i < Rq / 2; ++i) {
                zA[i] = a_[i];
                zA[Rq / 2 + i] = b_[i];
                zB[i] = b_[Rq / 2 + i];
            }
#pragma unroll
            for (int j = Rq / 2; j < Rq - 1; ++j) zB[j] = a_[j + 1];
            zB[Rq - 1] = a_[0];
        }

        float2 base = make_float2(1.f, 0.f), base2 = make_float2(1.f, 0.f);
        if (prm.per_spectrum) {
            auto E_of = [&](int k) {                      // exp(i phi) exp(-2 pi i d_eff k / N), d_eff = d + cr
                const double t = -d_eff_turn_scale * (double)k - (double)((cr * k) & (N - 1)) / (double)N;
                return cmulf(phasor_turns(t), sph->ephi);
            };
            base = E_of(pidx);
            if (special) base2 = E_of(Q / 2);
        }

        float *yout = nullptr;
        uint32_t *rec = nullptr;
        if (F32OUT) yout = prm.out_f32 + (((int64_t)a * prm.n_spectra + m) * n) * 4 + p * 2;
        else rec = reinterpret_cast<uint32_t *>(prm.out + (((int64_t)a * prm.n_spectra + m) * n) * 4);

#pragma unroll
        for (int kq = 0; kq < Rq; ++kq) {
            const int kA = special ? (kq < Rq / 2 ? Q * kq : Q / 2 + Q * (kq - Rq / 2)) : pidx + Q * kq;
            const int kB = n - kA;                        // == n for the DC pair (dropped Nyquist)
            const cx<float> zk = zA[kq], zm = zB[Rq - 1 - kq];
            const float2 tp = __ldg(tpost + kA);          // i w^k = (sin, cos)(2 pi k / N)
            const float sr = zk.re + zm.re, si = zk.im - zm.im;     // S = Z[k] + conj Z[n-k]
            const float dr = zk.re - zm.re, di = zk.im + zm.im;     // D = Z[k] - conj Z[n-k]
            const float fr = fmaf(-di, tp.y, dr * tp.x);            // F = D * (i w^k)
            const float fi = fmaf(di, tp.x, dr * tp.y);
            const float xkr = sr - fr, xki = si - fi;               // 2 X[k]
            const float xmr = sr + fr, xmi = -(si + fi);            // 2 X[n-k] = conj(S + F)
            float2 rgA, rgB;
            if (prm.per_spectrum) {
                const bool hi = special && kq >= Rq / 2;
                const float2 stp = sph->step[hi ? kq - Rq / 2 : kq];
                const float2 E = cmulf(hi ? base2 : base, stp);
                const float2 gA = __ldg(gtab + kA);
                const float2 gB = __ldg(gtab + (kB & (n - 1)));
                rgA = cmulf(E, gA);
                rgB = cmulf(cmulf(sph->c3, make_float2(E.x, -E.y)), gB);
                rgA.x *= 0.5f; rgA.y *= 0.5f; rgB.x *= 0.5f; rgB.y *= 0.5f;
            } else {
                rgA = __ldg(gtab + kA);
                rgB = __ldg(gtab + (kB & (n - 1)));
            }
            const float yAr = fmaf(-xki, rgA.y, xkr * rgA.x), yAi = fmaf(xki, rgA.x, xkr * rgA.y);
            const float yBr = fmaf(-xmi, rgB.y, xmr * rgB.x), yBi = fmaf(xmi, rgB.x, xmr * rgB.y);
            if (F32OUT) {
                *reinterpret_cast<float2 *>(yout + (int64_t)kA * 4) = make_float2(yAr, yAi);
                if (kB < n) *reinterpret_cast<float2 *>(yout + (int64_t)kB * 4) = make_float2(yBr, yBi);
            } else {
                // lane p = 0 stores channel kA, lane p = 1 channel kB; each fetches the other pol from its neighbour
                const uint32_t qA = quantize_pair(yAr, yAi), qB = quantize_pair(yBr, yBi);
                const uint32_t other = __shfl_xor_sync(0xffffffffu, p ? qA : qB, 1);
                if (p == 0) rec[kA] = __byte_perm(qA, other, 0x5410);            // {re0, im0, re1, im1}
                else if (kB < n) rec[kB] = __byte_perm(other, qB, 0x5410);
            }
        }
        if ((it & ~31) == 0) {                            // channel n/2: X = conj Z[n/2] (special lanes; warp-uniform branch)
            float2 rg;
            if (prm.per_spectrum) {
                const float2 E = cmulf(sph->ephi, sph->step[Rq / 2]);   // k = Q * Rq/2 = n/2
                rg = cmulf(E, __ldg(gtab + n / 2));
            } else {
                const float2 t = __ldg(gtab + n / 2);
                rg = make_float2(2.f * t.x, 2.f * t.y);                // table holds 0.5 * ...
            }
            const float xr = zhalf.re, xi = -zhalf.im;
            const float yr = fmaf(-xi, rg.y, xr * rg.x), yi = fmaf(xi, rg.x, xr * rg.y);
            if (F32OUT) {
                if (special) *reinterpret_cast<float2 *>(yout + (int64_t)(n / 2) * 4) = make_float2(yr, yi);
            } else {
                const uint32_t qh = quantize_pair(yr, yi);
                const uint32_t other = __shfl_xor_sync(0xffffffffu, qh, 1);
                if (special && p == 0) rec[n / 2] = __byte_perm(qh, other, 0x5410);
            }
        }
    }
}

template <class Plan>
constexpr size_t fft2_smem_bytes()
{
    return (size_t)Plan::units * 16 + 2 * sizeof(SpectrumPhase);
}

// One CTA per (antenna, spectrum), both pols.
template <class Plan, bool F32OUT>
__global__ void __launch_bounds__(Plan::tpf, (512 / Plan::tpf) > 0 ? (512 / Plan::tpf) : 1) fft2_kernel(const Fft2Params prm)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int n = Plan::n, N = 2 * n;
    float4 *sm = reinterpret_cast<float4 *>(smem_raw);
    SpectrumPhase *sph = reinterpret_cast<SpectrumPhase *>(smem_raw + (size_t)Plan::units * 16);

    const int tid = threadIdx.x;
    const int a = blockIdx.y;
    const int64_t m = prm.m_begin + blockIdx.x;
    if (m >= prm.m_end) return;

    const float4 *grow = reinterpret_cast<const float4 *>(prm.g + ((int64_t)a * prm.chunk_cap + (m - prm.m_begin)) * (int64_t)N * 2);

    double dts[2] = {0.0, 0.0};
    int cr[2] = {0, 0};
    if (prm.per_spectrum) {
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            const int64_t st = (int64_t)a * 2 + p;
            const int32_t c = prm.coarse[st * prm.n_coarse + (prm.n_coarse == 1 ? 0 : m)];
            cr[p] = (int)(c & (N - 1));
            const double d = (double)prm.fine_d[st * prm.n_fine + (prm.n_fine == 1 ? 0 : m)];
            const double phi = (double)prm.fine_phi[st * prm.n_fine + (prm.n_fine == 1 ? 0 : m)];
            dts[p] = d / (double)N;
            const int t = tid - 32 * p;                   // warp p sets up pol p
            if (t >= 0 && t < 16) {
                const int k = Plan::Q * t;
                const double tt = -dts[p] * (double)k - (double)((cr[p] * k) & (N - 1)) / (double)N;
                sph[p].step[t] = phasor_turns(tt);
            } else if (t == 16) {
                double s, c_;
                sincos(phi, &s, &c_);
                sph[p].ephi = make_float2((float)c_, (float)s);
                sincos(2.0 * phi, &s, &c_);
                const float2 e2 = make_float2((float)c_, (float)s);
                float2 h = phasor_turns(-0.5 * d);        // exp(-i pi d_eff) = exp(-i pi d) * (-1)^cr
                if (cr[p] & 1) { h.x = -h.x; h.y = -h.y; }
                sph[p].c3 = cmulf(e2, h);
            }
        }
    }

    fft2_pass1<Plan>(grow, sm, prm.tw1, tid);
    __syncthreads();
    fft2_pass2<Plan>(sm, prm.tw2, tid);
    __syncthreads();
    fft2_pass3<Plan, F32OUT>(sm, prm, a, m, tid, sph, dts, cr);
}

// scalar twiddle table of one pass: tw[k][x] = W_M^{k x} = (cos, -sin)(2 pi k x / M)
__global__ void build_scalar_twiddles(float2 *tw, int R, int S, int M)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= R * S) return;
    const int k = idx / S, x = idx - k * S;
    double s, c;
    sincospi(-2.0 * (double)((k * x) % M) / (double)M, &s, &c);
    tw[idx] = make_float2((float)c, (float)s);
}

// debug: natural-order FIR output g [A][2][S][N] from pol-packed scratch rows (a*cap + m), undoing the rotation
__global__ void unrotate2_kernel(const float *gp, float *g_out, const int32_t *coarse, int64_t n_coarse,
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
