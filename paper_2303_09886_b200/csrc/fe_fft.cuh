// fe_fft.cuh -- steps 4-7 of the path: N-point real-to-complex FFT (keep n channels, drop Nyquist,
// PAPER.md:37), fine-delay rotation, bandpass gain, quantisation to
// int8 Gaussian integers with both polarisations interleaved.
//
// Method.  The real transform of length N = 2n is done as an n-point complex FFT of
// z[i] = g[2i] + i g[2i+1] followed by a post-twiddle (the technique PAPER.md:179-185 describes and
// merges into its post-processing kernel); here the whole FFT, the post-twiddle, the rotation, the
// gain and the quantisation are ONE kernel, one CTA per (antenna, spectrum), both pols in the CTA.
//
// n = R1*R2*..*Rq (q = 3 or 4 passes, radices 4/8/16).  Decimation in frequency, natural-order input:
//   pass p transforms digit p (t_p -> k_p) and multiplies by W_{M_{p-1}}^{k_p * tau'} where
//   M_{p-1} = R_p*..*R_q and tau' is the natural index of the not-yet-transformed digits;
//   output channel k = k1 + R1 k2 + R1 R2 k3 (+ ...).
// Passes 1..q-1 hold TWO adjacent points (tau', tau'+1) in the two lanes of packed FP32 registers
// (FFMA2/FADD2/FMUL2) and exchange through shared memory IN PLACE (a thread writes back exactly the
// units it read, so one __syncthreads per pass); a 16-byte unit is {re0, re1, im0, im1}.
// The last pass is scalar: a thread transforms residue K and its mirror Q-K (Q = n/Rq) so that it
// owns both Z[k] and Z[n-k] and can do the real-FFT post-twiddle without another exchange (the
// paper's kernel likewise ran "two such FFTs ... by the same thread").
//
// The rotation phasor also carries the sub-row part cr of the coarse delay: the FIR kernel wrote
// the row circularly shifted by cr (fe_fir.cuh), so X[k] = exp(-2 pi i k cr/N) FFT(g')[k].
#pragma once
#include "fe_common.cuh"

namespace fe {

// ------------------------------------------------------------------------------------------------
// compile-time twiddles of the in-register butterflies: W_32^j = cos(2 pi j/32) - i sin(2 pi j/32)
// ------------------------------------------------------------------------------------------------
__host__ __device__ constexpr float w32_cos(int j)
{
    constexpr float c[9] = {1.0f, 0.98078528040323043f, 0.92387953251128674f, 0.83146961230254524f,
                            0.70710678118654752f, 0.55557023301960218f, 0.38268343236508977f,
                            0.19509032201612825f, 0.0f};
    j &= 31;
    if (j <= 8) return c[j];
    if (j <= 16) return -c[16 - j];
    if (j <= 24) return -c[j - 16];
    return c[32 - j];
}
__host__ __device__ constexpr float w32_sin(int j) { return w32_cos(j - 8); }   // sin(x) = cos(x - pi/2)

// x *= W_R^j  (forward transform: e^{-2 pi i j / R}), j, R compile-time
template <int R, int J, typename V>
__device__ __forceinline__ cx<V> mul_w(cx<V> x)
{
    constexpr int j32 = (J * (32 / R)) & 31;
    if constexpr (j32 == 0) {
        return x;
    } else if constexpr (j32 == 8) {            // -i
        return {x.im, -x.re};
    } else if constexpr (j32 == 16) {           // -1
        return {-x.re, -x.im};
    } else if constexpr (j32 == 24) {           // +i
        return {-x.im, x.re};
    } else if constexpr (j32 == 4) {            // (1 - i)/sqrt2
        constexpr float s = 0.70710678118654752f;
        return {(x.re + x.im) * s, (x.im - x.re) * s};
    } else if constexpr (j32 == 12) {           // (-1 - i)/sqrt2
        constexpr float s = 0.70710678118654752f;
        return {(x.im - x.re) * s, -((x.re + x.im) * s)};
    } else {
        constexpr float wr = w32_cos(j32), wi = -w32_sin(j32);
        return cmul(x, wr, wi);
    }
}

// In-register radix-R DIF butterfly, natural order in and out (R = 2, 4, 8, 16).
template <int R, typename V>
struct Dif {
    template <int J>
    static __device__ __forceinline__ void twiddle_half(cx<V> (&a)[R / 2], cx<V> (&b)[R / 2], const cx<V> (&x)[R])
    {
        if constexpr (J < R / 2) {
            a[J] = cadd(x[J], x[J + R / 2]);
            b[J] = mul_w<R, J, V>(csub(x[J], x[J + R / 2]));
            twiddle_half<J + 1>(a, b, x);
        }
    }
    static __device__ __forceinline__ void run(cx<V> (&x)[R])
    {
        if constexpr (R == 2) {
            const cx<V> a = cadd(x[0], x[1]), b = csub(x[0], x[1]);
            x[0] = a;
            x[1] = b;
        } else {
            cx<V> a[R / 2], b[R / 2];
            twiddle_half<0>(a, b, x);
            Dif<R / 2, V>::run(a);
            Dif<R / 2, V>::run(b);
#pragma unroll
            for (int k = 0; k < R / 2; ++k) {
                x[2 * k] = a[k];
                x[2 * k + 1] = b[k];
            }
        }
    }
};

// ------------------------------------------------------------------------------------------------
// FFT plan (compile time)
// ------------------------------------------------------------------------------------------------
template <int N_CH, int NPASS, int R1, int R2, int R3, int R4, int TPF, int SWEEPS = 1>
struct FftPlan {
    static constexpr int n = N_CH;
    static constexpr int q = NPASS;
    static constexpr int tpf = TPF;                       // threads per pol-FFT
    // SWEEPS = 2 (n = 32768, whose 256 KiB working set exceeds one SM's shared memory): the first
    // pass is a radix-R1 butterfly of which sweep h keeps only the outputs k1 = h (mod 2), i.e. the
    // top radix-2 stage of the decimation in frequency splits the transform into two independent
    // n/2-point halves (even / odd channels) that go through the exchange buffer one after the other.
    static constexpr int sweeps = SWEEPS;
    static_assert(SWEEPS == 1 || SWEEPS == 2, "1 or 2 sweeps");
    static_assert(SWEEPS == 1 || R1 % 2 == 0, "two sweeps need an even first radix");
    static_assert(NPASS == 3 || NPASS == 4, "3 or 4 passes");
    static_assert(R1 * R2 * R3 * R4 == N_CH, "radices must multiply to n");
    static_assert(NPASS == 4 || R4 == 1, "R4 unused with 3 passes");
    __host__ __device__ static constexpr int radix(int p) { return p == 1 ? R1 : p == 2 ? R2 : p == 3 ? R3 : R4; }
    static constexpr int Rq = NPASS == 3 ? R3 : R4;
    static constexpr int Q = N_CH / Rq;                   // residues handled by the last pass
    static constexpr int units = N_CH / 2 / SWEEPS;       // 16-byte units in the exchange buffer
    // M_p = R_{p+1} * ... * R_q  (M_0 = n)
    __host__ __device__ static constexpr int M(int p)
    {
        int m = N_CH;
        for (int i = 1; i <= p; ++i) m /= radix(i);
        return m;
    }
    // stride (in units) of digit p in the in-place layout [d1][d2]..[d_{q-1}][pair]
    __host__ __device__ static constexpr int S(int p) { return M(p) / 2; }
};

// unit address swizzle: XOR the low 3 bits with the low 3 bits of digit 1 (conflict-free 128-bit
// accesses both for "8 consecutive pair indices" (passes 1..q-1) and "8 consecutive k1" (last pass))
// Plans whose third pass has a stride of 4 units (n = 16384, 32768) would see units 32 apart (the same banks) in one
// quarter-warp of that pass; XORing bit 5 into bit 2 removes that 2-way conflict at the price of a 1.1-way one on the
// last pass's loads (checked for every plan and pass with a host-side model of the bank mapping).
template <class Plan>
__device__ __forceinline__ int swz(int lin)
{
    const int d1 = lin / Plan::S(1);
    int s = lin ^ (d1 & 7);
    if constexpr (Plan::q == 4 && Plan::S(3) == 4) s ^= ((lin >> 5) & 1) << 2;
    return s;
}

struct FftTables {
    const float4 *tw[3];      // pass p (1..q-1): [R_p][S(p)] {wr(2lo), wr(2lo+1), wi(2lo), wi(2lo+1)} of W_{M(p-1)}^{k tau'}
    const float2 *tpost;      // [n] (sin, cos)(2 pi k / N)  =  i * exp(-2 pi i k / N)
};

struct FftParams {
    const float *g;           // scratch rows, (a*chunk_cap + (m - m_begin))*P + p
    int8_t *out;              // [A][S][n][P][2] or null
    float *out_f32;           // [A][S][n][P][2] or null
    FftTables tab;
    const float2 *rg;         // const mode: [A][P][n]  0.5 * G * exp(i(-2 pi (d + cr) k/N + phi))
    const float2 *gains;      // per-spectrum mode: [A][P][n]
    const int32_t *coarse;    // [A*P][n_coarse]
    const float *fine_d;      // [A*P][n_fine]
    const float *fine_phi;    // [A*P][n_fine]
    int64_t n_coarse, n_fine;
    int64_t m_begin, m_end, chunk_cap, n_spectra;
    int P;
    int per_spectrum;         // 1: phasors computed in-kernel from the tables above
};

// ---- pass 1: global (scratch g') -> butterfly -> twiddle -> shared ---------------------------------
// Pass twiddles W^{k x}, k = 1..R-1, as running powers of the one table word W^{x} (both packed lanes hold their own
// x): the table walk of R-1 float4 words per butterfly (64 KB per spectrum in pass 1 of n = 8192) becomes one word,
// which keeps the L1 for the gain table.  The running product adds at most R rounding steps (< 2e-6 relative).
__device__ __forceinline__ cx<f2> cmulp(cx<f2> a, cx<f2> b)
{
    return {fnma_(a.im, b.im, a.re * b.re), fma_(a.im, b.re, a.re * b.im)};
}
__device__ __forceinline__ cx<f2> load_tw(const float4 *__restrict__ p)
{
    const float4 w = __ldg(p);
    return {f2(w.x, w.y), f2(w.z, w.w)};
}

template <class Plan>
__device__ __forceinline__ void fft_pass_first(const float4 *__restrict__ grow, float4 *sm, const float4 *__restrict__ tw,
                                               int tid)
{
    constexpr int R = Plan::radix(1);
    constexpr int ncol = Plan::S(1);                      // n / (2 R1) column pairs
    for (int col = tid; col < ncol; col += Plan::tpf) {
        cx<f2> x[R];
#pragma unroll
        for (int t = 0; t < R; ++t) {
            const float4 v = ldg_stream_f4(grow + t * ncol + col);
            x[t].re = f2(v.x, v.y);
            x[t].im = f2(v.z, v.w);
        }
        const cx<f2> w1 = load_tw(tw + ncol + col);
        Dif<R, f2>::run(x);
        cx<f2> wk = w1;
#pragma unroll
        for (int k = 0; k < R; ++k) {
            cx<f2> y = x[k];
            if (k > 0) {
                y = cmulp(x[k], wk);
                if (k + 1 < R) wk = cmulp(wk, w1);
            }
            sm[swz<Plan>(k * ncol + col)] = make_float4(y.re.v.x, y.re.v.y, y.im.v.x, y.im.v.y);
        }
    }
}

// top radix-2 stage of a two-sweep first pass, element J (compile-time recursion so that W_R1^J is constant)
template <class Plan, int H, int J>
__device__ __forceinline__ void sweep_half(const float4 *__restrict__ grow, int col, cx<f2> (&a)[Plan::radix(1) / 2])
{
    constexpr int R = Plan::radix(1), RH = R / 2;
    constexpr int ncol = Plan::S(1);
    if constexpr (J < RH) {
        const float4 u = ldg_stream_f4(grow + J * ncol + col);
        const float4 v = ldg_stream_f4(grow + (J + RH) * ncol + col);
        const cx<f2> xu = {f2(u.x, u.y), f2(u.z, u.w)}, xv = {f2(v.x, v.y), f2(v.z, v.w)};
        if constexpr (H == 0)
            a[J] = cadd(xu, xv);
        else
            a[J] = mul_w<R, J, f2>(csub(xu, xv));
        sweep_half<Plan, H, J + 1>(grow, col, a);
    }
}

// ---- pass 1 of a two-sweep plan: sweep H keeps the outputs k1 = 2 k'' + H of the radix-R1 butterfly.
// Its top radix-2 stage is a[j] = x[j] + x[j + R1/2] (H = 0) or (x[j] - x[j + R1/2]) W_R1^j (H = 1);
// the radix-R1/2 butterfly of a then gives k'' in natural order.  The row is read once per sweep.
template <class Plan, int H>
__device__ __forceinline__ void fft_pass_first_sweep(const float4 *__restrict__ grow, float4 *sm,
                                                     const float4 *__restrict__ tw, int tid)
{
    constexpr int R = Plan::radix(1), RH = R / 2;
    constexpr int ncol = Plan::S(1);
    for (int col = tid; col < ncol; col += Plan::tpf) {
        cx<f2> a[RH];
        const cx<f2> w1 = load_tw(tw + ncol + col);        // W^{x}; outputs need W^{(2 kk + H) x}
        sweep_half<Plan, H, 0>(grow, col, a);
        Dif<RH, f2>::run(a);
        const cx<f2> w2 = cmulp(w1, w1);
        cx<f2> wk = H ? w1 : w2;                           // first non-trivial twiddle: k1 = 1 (H = 1) or 2 (H = 0)
#pragma unroll
        for (int kk = 0; kk < RH; ++kk) {
            const int k1 = 2 * kk + H;
            cx<f2> y = a[kk];
            if (k1 > 0) {
                y = cmulp(a[kk], wk);
                if (kk + 1 < RH) wk = cmulp(wk, w2);
            }
            sm[swz<Plan>(kk * ncol + col)] = make_float4(y.re.v.x, y.re.v.y, y.im.v.x, y.im.v.y);
        }
    }
}

// ---- middle pass p: shared -> butterfly -> twiddle -> shared (in place) -----------------------------
template <class Plan, int PASS>
__device__ __forceinline__ void fft_pass_mid(float4 *sm, const float4 *__restrict__ tw, int tid)
{
    constexpr int R = Plan::radix(PASS);
    constexpr int Sp = Plan::S(PASS);                     // stride of digit PASS, = number of "lo" values
    constexpr int ncol = Plan::units / R;
    for (int col = tid; col < ncol; col += Plan::tpf) {
        const int hi = col / Sp, lo = col - hi * Sp;
        const int base = hi * (R * Sp) + lo;
        cx<f2> x[R];
#pragma unroll
        for (int t = 0; t < R; ++t) {
            const float4 v = sm[swz<Plan>(base + t * Sp)];
            x[t].re = f2(v.x, v.y);
            x[t].im = f2(v.z, v.w);
        }
        const cx<f2> w1 = load_tw(tw + Sp + lo);
        Dif<R, f2>::run(x);
        cx<f2> wk = w1;
#pragma unroll
        for (int k = 0; k < R; ++k) {
            cx<f2> y = x[k];
            if (k > 0) {
                y = cmulp(x[k], wk);
                if (k + 1 < R) wk = cmulp(wk, w1);
            }
            sm[swz<Plan>(base + k * Sp)] = make_float4(y.re.v.x, y.re.v.y, y.im.v.x, y.im.v.y);
        }
    }
}

// storage index (in units, before the pair index) of residue K = k1 + R1 k2 + R1 R2 k3
template <class Plan>
__device__ __forceinline__ int residue_to_store(int K)
{
    int store = 0, rem = K;
#pragma unroll
    for (int p = 1; p < Plan::q; ++p) {
        const int r = Plan::radix(p);
        int d = rem % r;
        rem /= r;
        if (p == 1) d /= Plan::sweeps;                    // two sweeps: the buffer holds k1 = 2 d + h
        store = store * r + d;
    }
    return store;
}

template <class Plan>
__device__ __forceinline__ void fft_load_residue(const float4 *sm, int K, cx<float> (&z)[Plan::Rq])
{
    const int base = residue_to_store<Plan>(K) * (Plan::Rq / 2);
#pragma unroll
    for (int c = 0; c < Plan::Rq / 2; ++c) {
        const float4 v = sm[swz<Plan>(base + c)];
        z[2 * c] = {v.x, v.z};
        z[2 * c + 1] = {v.y, v.w};
    }
    Dif<Plan::Rq, float>::run(z);
}

__device__ __forceinline__ uint32_t quantize_pair(float re, float im)
{
    // round-half-even + clamp to [-127, 127] ("rounding and saturation"): the FP32 add
    // of 1.5*2^23 rounds to nearest-even and leaves the integer in the low mantissa bits.
    const float magic = 12582912.0f;
    const float r = fminf(fmaxf(re, -127.0f), 127.0f) + magic;
    const float i = fminf(fmaxf(im, -127.0f), 127.0f) + magic;
    return __byte_perm(__float_as_uint(r), __float_as_uint(i), 0x0040);   // byte0 = re, byte1 = im
}

// phasor helpers for the per-spectrum mode (float64 trigonometry, one call per thread per spectrum)
__device__ __forceinline__ float2 phasor_turns(double turns)
{
    double s, c;
    sincospi(2.0 * turns, &s, &c);
    return make_float2((float)c, (float)s);
}
__device__ __forceinline__ float2 cmulf(float2 a, float2 b)
{
    return make_float2(fmaf(-a.y, b.y, a.x * b.x), fmaf(a.y, b.x, a.x * b.y));
}

struct SpectrumPhase {       // shared, per pol: filled once per spectrum in per-spectrum mode
    float2 step[16];         // exp(-2 pi i d_eff Q kq / N)
    float2 c3;               // exp(2 i phi) exp(-i pi d_eff): R[n-k] = c3 * conj(E[k]) with E incl. exp(i phi)
    float2 ephi;             // exp(i phi)
};

// ---- last pass + post-twiddle + rotation + gain + quantise -----------------------------------------
template <class Plan, bool F32OUT>
__device__ __forceinline__ void fft_pass_last(const float4 *sm, const FftParams &prm, int a, int pol, int64_t m,
                                              int tid, uint16_t *stage, const SpectrumPhase *sph,
                                              double d_eff_turn_scale, int cr, int sweep)
{
    constexpr int Rq = Plan::Rq, Q = Plan::Q, n = Plan::n, N = 2 * n;
    const float2 *__restrict__ tpost = prm.tab.tpost;
    const int64_t st = (int64_t)a * prm.P + pol;
    const float2 *__restrict__ gtab = (prm.per_spectrum ? prm.gains : prm.rg) + st * n;
    float *yout = nullptr;
    if (F32OUT) yout = prm.out_f32 + (((int64_t)a * prm.n_spectra + m) * n) * prm.P * 2 + pol * 2;

    constexpr int SW = Plan::sweeps;
    for (int jdx = tid; jdx < Q / 2 / SW; jdx += Plan::tpf) {
        const int pidx = SW * jdx + sweep;                // residue K of this sweep's parity
        cx<float> zA[Rq], zB[Rq];
        const bool special = pidx == 0;
        fft_load_residue<Plan>(sm, pidx, zA);
        fft_load_residue<Plan>(sm, special ? Q / 2 : Q - pidx, zB);

        cx<float> zhalf = zA[Rq / 2];                     // only meaningful for the special thread
        if (special) {                                    // re-pair: see DESIGN.md section 6 ("mirror pairs")
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

        // per-spectrum mode: base phasor of this thread
        float2 base = make_float2(1.f, 0.f), base2 = make_float2(1.f, 0.f);
        if (prm.per_spectrum) {
            auto E_of = [&](int k) {                      // exp(i phi) exp(-2 pi i d_eff k / N), d_eff = d + cr
                const double t = -d_eff_turn_scale * (double)k - (double)((cr * k) & (N - 1)) / (double)N;
                return cmulf(phasor_turns(t), sph->ephi);
            };
            base = E_of(pidx);
            if (special) base2 = E_of(Q / 2);
        }

        // Table words are requested a group of GK channel pairs ahead of their use (one exposed L2 round trip per
        // group instead of one per pair), and the post-twiddle phasor of pair kq is the thread's own
        // (sin, cos)(2 pi K / N) rotated by the compile-time angle 2 pi kq Q / N = 2 pi kq / (2 Rq).
        constexpr int GK = 4;
        const float2 tpK = __ldg(tpost + pidx);
        float2 gAq[GK], gBq[GK];
        auto k_of = [&](int kq) { return special ? (kq < Rq / 2 ? Q * kq : Q / 2 + Q * (kq - Rq / 2)) : pidx + Q * kq; };
#pragma unroll
        for (int kq = 0; kq < Rq; ++kq) {
            if (kq % GK == 0) {
#pragma unroll
                for (int g = 0; g < GK; ++g) {
                    const int kAg = k_of(kq + g);
                    gAq[g] = __ldg(gtab + kAg);
                    gBq[g] = __ldg(gtab + ((n - kAg) & (n - 1)));
                }
            }
            const int kA = k_of(kq);
            const int kB = n - kA;                        // == n for the DC pair (dropped Nyquist)
            const cx<float> zk = zA[kq], zm = zB[Rq - 1 - kq];
            float2 tp;                                    // i w^k = (sin, cos)(2 pi k / N)
            if (special) {
                tp = __ldg(tpost + kA);
            } else {
                constexpr int st = 32 / (2 * Rq);
                const float cphi = w32_cos(kq * st), sphi = w32_sin(kq * st);
                tp = make_float2(fmaf(tpK.x, cphi, tpK.y * sphi), fmaf(-tpK.x, sphi, tpK.y * cphi));
            }
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
                const float2 gA = gAq[kq % GK];
                const float2 gB = gBq[kq % GK];
                rgA = cmulf(E, gA);
                rgB = cmulf(cmulf(sph->c3, make_float2(E.x, -E.y)), gB);
                rgA.x *= 0.5f; rgA.y *= 0.5f; rgB.x *= 0.5f; rgB.y *= 0.5f;
            } else {
                rgA = gAq[kq % GK];
                rgB = gBq[kq % GK];
            }
            const float yAr = fmaf(-xki, rgA.y, xkr * rgA.x), yAi = fmaf(xki, rgA.x, xkr * rgA.y);
            const float yBr = fmaf(-xmi, rgB.y, xmr * rgB.x), yBi = fmaf(xmi, rgB.x, xmr * rgB.y);
            if (F32OUT) {
                *reinterpret_cast<float2 *>(yout + (int64_t)kA * prm.P * 2) = make_float2(yAr, yAi);
                if (kB < n) *reinterpret_cast<float2 *>(yout + (int64_t)kB * prm.P * 2) = make_float2(yBr, yBi);
            } else {
                stage[(kA / SW) * prm.P + pol] = (uint16_t)quantize_pair(yAr, yAi);
                if (kB < n) stage[(kB / SW) * prm.P + pol] = (uint16_t)quantize_pair(yBr, yBi);
            }
        }
        if (special) {                                    // channel n/2: X = conj Z[n/2]
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
            if (F32OUT)
                *reinterpret_cast<float2 *>(yout + (int64_t)(n / 2) * prm.P * 2) = make_float2(yr, yi);
            else
                stage[(n / 2 / SW) * prm.P + pol] = (uint16_t)quantize_pair(yr, yi);
        }
    }
}

template <class Plan>
constexpr size_t fft_smem_bytes(int P)
{
    return (size_t)Plan::units * 16 + (size_t)(Plan::n / Plan::sweeps) * P * 2 + sizeof(SpectrumPhase);
}

// One CTA per (antenna, spectrum); the pols are transformed one after the other through the same
// exchange buffer (small CTAs, several per SM, each at a different phase of its spectrum).  A
// two-sweep plan (n = 32768) runs the whole sequence once for the even and once for the odd channels.
template <class Plan, bool F32OUT>
static __global__ void __launch_bounds__(Plan::tpf, (512 / Plan::tpf) > 0 ? (512 / Plan::tpf) : 1) fft_kernel(const FftParams prm)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int n = Plan::n, N = 2 * n, SW = Plan::sweeps;
    const int P = prm.P;
    float4 *sm = reinterpret_cast<float4 *>(smem_raw);
    uint16_t *stage = reinterpret_cast<uint16_t *>(smem_raw + (size_t)Plan::units * 16);
    SpectrumPhase *sph = reinterpret_cast<SpectrumPhase *>(smem_raw + (size_t)Plan::units * 16 + (size_t)(n / SW) * P * 2);

    const int tid = threadIdx.x;
    // reverse of the FIR kernel's write order: the newest scratch rows are still in L2 (see fft2_kernel)
    const int a = (int)gridDim.y - 1 - (int)blockIdx.y;
    const int64_t m = prm.m_end - 1 - (int64_t)blockIdx.x;
    if (m < prm.m_begin) return;

    for (int sweep = 0; sweep < SW; ++sweep) {
        for (int pol = 0; pol < P; ++pol) {
            const int64_t st = (int64_t)a * P + pol;
            const float4 *grow = reinterpret_cast<const float4 *>(
                prm.g + (((int64_t)a * prm.chunk_cap + (m - prm.m_begin)) * P + pol) * (int64_t)N);

            // per-spectrum phasor set-up
            double dts = 0.0;
            int cr = 0;
            if (prm.per_spectrum) {
                const int32_t c = prm.coarse[st * prm.n_coarse + (prm.n_coarse == 1 ? 0 : m)];
                cr = (int)(c & (N - 1));
                const double d = (double)prm.fine_d[st * prm.n_fine + (prm.n_fine == 1 ? 0 : m)];
                const double phi = (double)prm.fine_phi[st * prm.n_fine + (prm.n_fine == 1 ? 0 : m)];
                dts = d / (double)N;                      // turns per channel of the fractional part
                if (tid < 16) {
                    const int k = Plan::Q * tid;
                    const double t = -dts * (double)k - (double)((cr * k) & (N - 1)) / (double)N;
                    sph->step[tid] = phasor_turns(t);
                } else if (tid == 16) {
                    double s, c_;
                    sincos(phi, &s, &c_);
                    sph->ephi = make_float2((float)c_, (float)s);
                    sincos(2.0 * phi, &s, &c_);
                    const float2 e2 = make_float2((float)c_, (float)s);
                    float2 h = phasor_turns(-0.5 * d);    // exp(-i pi d_eff) = exp(-i pi d) * (-1)^cr
                    if (cr & 1) { h.x = -h.x; h.y = -h.y; }
                    sph->c3 = cmulf(e2, h);
                }
            }

            if constexpr (SW == 1) {
                fft_pass_first<Plan>(grow, sm, prm.tab.tw[0], tid);
            } else {
                if (sweep == 0)
                    fft_pass_first_sweep<Plan, 0>(grow, sm, prm.tab.tw[0], tid);
                else
                    fft_pass_first_sweep<Plan, 1>(grow, sm, prm.tab.tw[0], tid);
            }
            __syncthreads();
            fft_pass_mid<Plan, 2>(sm, prm.tab.tw[1], tid);
            __syncthreads();
            if constexpr (Plan::q == 4) {
                fft_pass_mid<Plan, 3>(sm, prm.tab.tw[2], tid);
                __syncthreads();
            }
            fft_pass_last<Plan, F32OUT>(sm, prm, a, pol, m, tid, stage, sph, dts, cr, sweep);
            if (pol + 1 < P || sweep + 1 < SW) __syncthreads();   // exchange buffer and phasors are reused
        }
        if (!F32OUT) {
            __syncthreads();
            int8_t *rec = prm.out + (((int64_t)a * prm.n_spectra + m) * n) * P * 2;
            if constexpr (SW == 1) {
                // coalesced copy-out of the staged record [n][P][2] int8
                const int n_vec = n * P * 2 / 16;
                uint4 *dst = reinterpret_cast<uint4 *>(rec);
                const uint4 *src = reinterpret_cast<const uint4 *>(stage);
                for (int i = threadIdx.x; i < n_vec; i += blockDim.x) stg_stream_u4(dst + i, src[i]);
            } else {
                // the stage holds the channels k = SW i + sweep: [n / SW][P][2] int8, one P*2-byte group each
                if (P == 2) {
                    const uint32_t *src = reinterpret_cast<const uint32_t *>(stage);
                    uint32_t *dst = reinterpret_cast<uint32_t *>(rec);
                    for (int i = threadIdx.x; i < n / SW; i += blockDim.x) dst[SW * i + sweep] = src[i];
                } else {
                    uint16_t *dst = reinterpret_cast<uint16_t *>(rec);
                    for (int i = threadIdx.x; i < n / SW; i += blockDim.x) dst[SW * i + sweep] = stage[i];
                }
                if (sweep + 1 < SW) __syncthreads();      // stage is reused by the next sweep
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// table builders (device, float64 trigonometry; run once at create / when parameters change)
// ------------------------------------------------------------------------------------------------
// tw[k][lo] for one pass: W_M^{k tau'}, tau' = 2 lo, 2 lo + 1
static __global__ void build_pass_twiddles(float4 *tw, int R, int S, int M)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= R * S) return;
    const int k = idx / S, lo = idx - k * S;
    double s0, c0, s1, c1;
    const int e0 = (k * (2 * lo)) % M, e1 = (k * (2 * lo + 1)) % M;
    sincospi(-2.0 * (double)e0 / (double)M, &s0, &c0);
    sincospi(-2.0 * (double)e1 / (double)M, &s1, &c1);
    tw[idx] = make_float4((float)c0, (float)c1, (float)s0, (float)s1);
}

static __global__ void build_post_twiddles(float2 *tp, int n)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    double s, c;
    sincospi((double)k / (double)n, &s, &c);              // 2 pi k / N = pi k / n
    tp[k] = make_float2((float)s, (float)c);
}

// const mode: rg[a][p][k] = 0.5 * G * exp(i(-2 pi (d + cr) k / N + phi))
static __global__ void build_rg_table(float2 *rg, const float2 *gains, const int32_t *coarse, const float *fine_d,
                               const float *fine_phi, int n, int n_streams)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int st = blockIdx.y;
    if (k >= n || st >= n_streams) return;
    const int N = 2 * n;
    const int cr = (int)(coarse[st] & (N - 1));
    const double d = (double)fine_d[st], phi = (double)fine_phi[st];
    const double turns = -d * (double)k / (double)N - (double)(((int64_t)cr * k) & (N - 1)) / (double)N;
    double s, c, sp, cp;
    sincospi(2.0 * turns, &s, &c);
    sincos(phi, &sp, &cp);
    const double rr = c * cp - s * sp, ri = c * sp + s * cp;
    const float2 g = gains[(int64_t)st * n + k];
    const double yr = 0.5 * ((double)g.x * rr - (double)g.y * ri);
    const double yi = 0.5 * ((double)g.x * ri + (double)g.y * rr);
    rg[(int64_t)st * n + k] = make_float2((float)yr, (float)yi);
}

}  // namespace fe
