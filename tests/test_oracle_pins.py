"""Pins for the float64 oracle (CPU only, `-m "not gpu"`).

Each test checks oracle/ against something OTHER than itself: a hand-derived value, a closed form,
an invariant, a library routine on a special case, or a brute-force numpy restatement of the
definition.  The pin numbers P1..P12 are those of SURVEY.md section 8(c) / DESIGN.md.
"""
from pathlib import Path

import numpy as np
import pytest

import oracle
import synth_inputs as si

GOLD = Path(__file__).resolve().parent / "golden"


def _golden_rows(name):
    rows = []
    for line in (GOLD / name).read_text().splitlines():
        line = line.strip()
        if line and not line.startswith("#"):
            rows.append(line)
    return rows


def brute_force(samples, n, T, h, c, d, phi, G, m):
    """The definition, written with numpy and nothing else (pin P12).

    X[k] = sum_{m'<NT} h[m'] s[N m - c + m'] exp(-2 pi i k m'/N), Y = X exp(i(-2 pi d k/N + phi)) G.
    """
    N = 2 * n
    idx = N * m - c + np.arange(N * T)
    ok = (idx >= 0) & (idx < samples.size)
    x = np.where(ok, samples[np.clip(idx, 0, samples.size - 1)], 0).astype(np.float64)
    k = np.arange(n)[:, None]
    mp = np.arange(N * T)[None, :]
    E = np.exp(-2j * np.pi * ((k * mp) % N) / N)
    X = E @ (x * h.astype(np.float64))
    kk = np.arange(n)
    R = np.exp(1j * (-2 * np.pi * float(np.float32(d)) * kk / N + float(np.float32(phi))))
    return X * R * G.astype(np.complex128)


# ------------------------------------------------------------------------------------------ P1
def test_p1_unpack_hand_example():
    (row,) = _golden_rows("pack_example.txt")
    left, right = row.split(":")
    samples = np.array([int(v) for v in left.split()], dtype=np.int16)
    packed = np.array([int(v, 16) for v in right.split()], dtype=np.uint8)
    np.testing.assert_array_equal(oracle.unpack10(packed, 4), samples)
    np.testing.assert_array_equal(si.pack10_bitwise(samples), packed)
    np.testing.assert_array_equal(si.pack10(samples), packed)


def test_p1_all_codes_roundtrip_through_independent_packer():
    codes = np.arange(-512, 512, dtype=np.int16)
    rng = np.random.default_rng(1)
    seq = np.concatenate([codes, rng.permutation(codes), codes[::-1]])
    packed = si.pack10_bitwise(seq)
    np.testing.assert_array_equal(oracle.unpack10(packed, seq.size), seq)
    np.testing.assert_array_equal(si.pack10(seq), packed)          # the fast generator packer agrees


def test_p1_single_bit_positions():
    # a walking one through 40 bits: each bit must land in exactly one sample at the MSB-first place
    for bit in range(40):
        b = np.zeros(5, dtype=np.uint8)
        b[bit >> 3] = 0x80 >> (bit & 7)
        s = oracle.unpack10(b, 4).astype(np.int64) & 0x3FF
        expect = np.zeros(4, dtype=np.int64)
        expect[bit // 10] = 1 << (9 - bit % 10)
        np.testing.assert_array_equal(s, expect)


# ------------------------------------------------------------------------------------------ P2
def test_p2_impulse_gives_weights():
    n, T, S = 8, 4, 6
    N = 2 * n
    rng = np.random.default_rng(2)
    h = rng.standard_normal(N * T).astype(np.float32)
    L = N * (S + T - 1)
    c = 5
    for ustar in (0, 7, 37, 100, L - 1):
        s = np.zeros(L)
        s[ustar] = 3.0
        for m in range(S):
            g = oracle.fir(oracle.window(s, N, T, m, c), h, N, T)
            expect = np.zeros(N)
            # N m - c + t + N j = ustar
            for j in range(T):
                t = ustar - N * m + c - N * j
                if 0 <= t < N:
                    expect[t] = 3.0 * float(h[t + N * j])
            np.testing.assert_allclose(g, expect, rtol=0, atol=0)


def test_p2_single_tap_is_block_fft():
    # T = 1, h = 1: the path is a plain block real FFT (library rfft as cross-check, never as oracle)
    n, S = 32, 5
    N = 2 * n
    rng = np.random.default_rng(3)
    s = rng.integers(-512, 512, size=(1, 1, N * S)).astype(np.float64)
    res = oracle.channelize_f64(s, n, 1, np.ones(N, dtype=np.float32))
    ref = np.fft.rfft(s.reshape(S, N), axis=1)[:, :n]
    np.testing.assert_allclose(res["Y"][0, :, :, 0], ref, rtol=0, atol=1e-9)


# ------------------------------------------------------------------------------------------ P3
def test_p3_coarse_delay_equals_zero_filled_shift():
    w = si.custom_workload(A=2, n=16, T=4, S=9, seed=4, random_weights=True)
    s = w.samples.astype(np.float64)
    for c in (1, 3, 17, 40, -6):
        coarse = np.full((w.A, w.P, 1), c, dtype=np.int32)
        a = oracle.channelize_f64(s, w.n, w.T, w.weights, coarse=coarse, gains=w.gains)
        shifted = np.zeros_like(s)
        if c >= 0:
            shifted[..., c:] = s[..., : s.shape[-1] - c]
        else:
            shifted[..., :c] = s[..., -c:]
        b = oracle.channelize_f64(shifted, w.n, w.T, w.weights, gains=w.gains)
        np.testing.assert_array_equal(a["Y"], b["Y"])          # bit-exact
        np.testing.assert_array_equal(a["out"], b["out"])


def test_p3_streams_are_independent():
    w = si.custom_workload(A=2, n=16, T=4, S=5, seed=5)
    s = w.samples.astype(np.float64)
    full = oracle.channelize_f64(s, w.n, w.T, w.weights, coarse=w.coarse, fine_delay=w.fine_delay,
                                 phase=w.phase, gains=w.gains)
    s2 = s.copy()
    s2[1, 0] = 0                                               # zero one stream
    part = oracle.channelize_f64(s2, w.n, w.T, w.weights, coarse=w.coarse, fine_delay=w.fine_delay,
                                 phase=w.phase, gains=w.gains)
    np.testing.assert_array_equal(full["Y"][0], part["Y"][0])
    np.testing.assert_array_equal(full["Y"][1, :, :, 1], part["Y"][1, :, :, 1])
    assert np.all(part["Y"][1, :, :, 0] == 0)


# ------------------------------------------------------------------------------------------ P4
@pytest.mark.parametrize("N", [2, 4, 8, 16, 64, 128])
def test_p4_fft_matches_quadratic_dft(N):
    rng = np.random.default_rng(N)
    g = rng.standard_normal(N)
    X_fft = oracle.fft_radix2(g + 0j)
    X_dft = oracle.dft(g)
    # and a third, numpy-written O(N^2) sum
    t = np.arange(N)
    X_np = np.array([np.sum(g * np.exp(-2j * np.pi * k * t / N)) for k in range(N)])
    np.testing.assert_allclose(X_fft, X_np, atol=1e-11)
    np.testing.assert_allclose(X_dft, X_np, atol=1e-11)


def test_p4_on_bin_tone_single_channel_and_sign():
    N, k0 = 256, 19
    t = np.arange(N)
    X = oracle.fft_radix2(np.cos(2 * np.pi * k0 * t / N + 0.3) + 0j)
    # forward sign e^{-i...}: the positive-frequency bin carries e^{+i theta} * N/2
    np.testing.assert_allclose(X[k0], N / 2 * np.exp(0.3j), atol=1e-9)
    np.testing.assert_allclose(X[N - k0], N / 2 * np.exp(-0.3j), atol=1e-9)
    mask = np.ones(N, bool)
    mask[[k0, N - k0]] = False
    assert np.abs(X[mask]).max() < 1e-9
    # complex exponential e^{+2 pi i k0 t/N} lands in bin k0 only (pins the sign of the exponent)
    Xc = oracle.fft_radix2(np.exp(2j * np.pi * k0 * t / N))
    assert abs(Xc[k0] - N) < 1e-9 and abs(Xc[N - k0]) < 1e-9


def test_p4_dc_bin_is_real():
    w = si.custom_workload(A=1, n=32, T=4, S=3, seed=6)
    res = oracle.channelize_f64(w.samples.astype(np.float64), w.n, w.T, w.weights)
    assert np.abs(res["Y"][..., 0, :].imag).max() < 1e-9


# ------------------------------------------------------------------------------------------ P5
def _Htilde(h, f):
    mp = np.arange(h.size)
    return np.sum(h.astype(np.float64) * np.exp(-2j * np.pi * f * mp))


@pytest.mark.parametrize("nu_bins", [100.0, 100.37, 3.5, 511.25])
def test_p5_tone_closed_form(nu_bins):
    # X[m,k] = (A/2)(e^{i(th + 2 pi nu u0)} H~(k/N - nu) + e^{-i(th + 2 pi nu u0)} H~(k/N + nu)), u0 = N m - c
    n, T, S = 512, 16, 4
    N = 2 * n
    h = si.hann_sinc_weights(n, T)
    amp, theta, c = 211.0, 0.7, 5
    nu = nu_bins / N
    L = N * (S + T - 1)
    u = np.arange(L)
    s = amp * np.cos(2 * np.pi * nu * u + theta)
    coarse = np.full((1, 1, 1), c, dtype=np.int32)
    res = oracle.channelize_f64(s.reshape(1, 1, L), n, T, h, coarse=coarse)
    for m in (1, 3):                                            # windows fully inside the batch
        u0 = N * m - c
        e = np.exp(1j * (theta + 2 * np.pi * nu * u0))
        for k in (0, 1, int(nu_bins) - 1, int(nu_bins), int(nu_bins) + 1, n - 1):
            if not 0 <= k < n:
                continue
            expect = amp / 2 * (e * _Htilde(h, k / N - nu) + np.conj(e) * _Htilde(h, k / N + nu))
            assert abs(res["Y"][0, m, k, 0] - expect) < 1e-7 * amp * N


def test_p5_hann_sinc_scale_and_leakage_match_survey_figures():
    (row,) = _golden_rows("hann_sinc_sums.txt")
    sum_h, sum_h2, leak1, leak2 = (float(v) for v in row.split())
    n, T = 1024, 16
    N = 2 * n
    h = si.hann_sinc_weights(n, T).astype(np.float64)
    assert abs(h.sum() / N - sum_h) < 2e-5
    assert abs((h ** 2).sum() / N - sum_h2) < 2e-5
    # on-bin tone through the oracle: neighbour leakage relative to the peak
    k0, amp = 100, 300.0
    L = N * (2 + T - 1)
    s = amp * np.cos(2 * np.pi * k0 * np.arange(L) / N)
    Y = oracle.channelize_f64(s.reshape(1, 1, L), n, T, h.astype(np.float32))["Y"][0, 0, :, 0]
    peak = abs(Y[k0])
    np.testing.assert_allclose(peak, amp / 2 * h.sum(), rtol=1e-6)
    assert abs(abs(Y[k0 + 1]) / peak - leak1) < 0.1 * leak1
    assert abs(abs(Y[k0 + 2]) / peak - leak2) < 0.15 * leak2


# ------------------------------------------------------------------------------------------ P6
def test_p6_parseval_with_nyquist():
    w = si.custom_workload(A=1, n=64, T=4, S=6, seed=7, random_weights=True)
    s = w.samples.astype(np.float64)
    res = oracle.channelize_f64(s, w.n, w.T, w.weights, want_nyq=True)
    N = w.N
    for p in range(2):
        for m in range(w.S):
            g = oracle.fir(oracle.window(s[0, p], N, w.T, m, 0), w.weights, N, w.T)
            X = res["Y"][0, m, :, p]
            nyq = res["nyquist"][0, p, m]
            rhs = (abs(X[0]) ** 2 + 2 * np.sum(np.abs(X[1:]) ** 2) + abs(nyq) ** 2) / N
            np.testing.assert_allclose(np.sum(g ** 2), rhs, rtol=1e-12)


# ------------------------------------------------------------------------------------------ P7
def test_p7_zero_fine_delay_unit_gain_is_identity_and_modulus():
    w = si.custom_workload(A=1, n=64, T=4, S=4, seed=8)
    s = w.samples.astype(np.float64)
    base = oracle.channelize_f64(s, w.n, w.T, w.weights)["Y"]
    same = oracle.channelize_f64(s, w.n, w.T, w.weights, fine_delay=np.zeros((1, 2, 1), np.float32),
                                 phase=np.zeros((1, 2, 1), np.float32),
                                 gains=np.ones((1, 2, w.n), np.complex64))["Y"]
    np.testing.assert_array_equal(base, same)
    rot = oracle.channelize_f64(s, w.n, w.T, w.weights, fine_delay=w.fine_delay, phase=w.phase,
                                gains=w.gains)["Y"]
    G = np.transpose(w.gains.astype(np.complex128), (0, 2, 1))[:, None]   # [A][1][n][P]
    np.testing.assert_allclose(np.abs(rot), np.abs(base) * np.abs(G), rtol=1e-12, atol=1e-12)
    # phase only: Y = X e^{i phi}
    ph = np.full((1, 2, 1), 0.3, np.float32)
    yphi = oracle.channelize_f64(s, w.n, w.T, w.weights, phase=ph)["Y"]
    np.testing.assert_allclose(yphi, base * np.exp(1j * float(np.float32(0.3))), rtol=1e-12, atol=1e-9)


def test_p7_integer_fine_delay_matches_coarse_delay_phase_on_tone():
    n, T, S, k0, c = 128, 8, 4, 37, 5
    N = 2 * n
    h = si.hann_sinc_weights(n, T)
    L = N * (S + T - 1)
    s = (200.0 * np.cos(2 * np.pi * k0 * np.arange(L) / N + 0.4)).reshape(1, 1, L)
    yc = oracle.channelize_f64(s, n, T, h, coarse=np.full((1, 1, 1), c, np.int32))["Y"][0, 2, k0, 0]
    yf = oracle.channelize_f64(s, n, T, h, fine_delay=np.full((1, 1, 1), float(c), np.float32))["Y"][0, 2, k0, 0]
    assert abs(yc - yf) < 1e-4 * abs(yc)
    # and the sign: a positive delay retards the phase of a positive-frequency tone
    y0 = oracle.channelize_f64(s, n, T, h)["Y"][0, 2, k0, 0]
    assert abs(yc / y0 - np.exp(-2j * np.pi * k0 * c / N)) < 1e-4


# ------------------------------------------------------------------------------------------ P8
def test_p8_linearity():
    rng = np.random.default_rng(9)
    n, T, S = 32, 4, 5
    N = 2 * n
    L = N * (S + T - 1)
    h = rng.standard_normal(N * T).astype(np.float32)
    s1 = rng.standard_normal((1, 2, L))
    s2 = rng.standard_normal((1, 2, L))
    kw = dict(coarse=np.array([[[3], [0]]], np.int32), fine_delay=np.full((1, 2, 1), 0.25, np.float32),
              phase=np.full((1, 2, 1), 0.1, np.float32),
              gains=(rng.standard_normal((1, 2, n)) + 1j * rng.standard_normal((1, 2, n))).astype(np.complex64))
    y1 = oracle.channelize_f64(s1, n, T, h, **kw)["Y"]
    y2 = oracle.channelize_f64(s2, n, T, h, **kw)["Y"]
    y12 = oracle.channelize_f64(2.5 * s1 - 0.75 * s2, n, T, h, **kw)["Y"]
    np.testing.assert_allclose(y12, 2.5 * y1 - 0.75 * y2, rtol=0, atol=1e-10 * np.abs(y12).max())


# ------------------------------------------------------------------------------------------ P9
def test_p9_quantize_table():
    for row in _golden_rows("quantize_table.txt"):
        v, q = row.split()
        assert oracle.quantize(float(v)) == int(q), row


def test_p9_saturation_through_the_path():
    # huge gain: every nonzero output clamps to +-127, never -128
    w = si.custom_workload(A=1, n=16, T=2, S=3, seed=10)
    res = oracle.process(w.packed, 1, w.n, w.T, 2, w.weights, w.S, gains=np.full((1, 2, w.n), 1e6, np.complex64))
    assert res["out"].min() == -127 and res["out"].max() == 127
    Yr = res["Y"].real
    assert np.all(res["out"][..., 0][np.abs(Yr.transpose(0, 1, 2, 3)) > 127.5] != 0)


# ------------------------------------------------------------------------------------------ P10
def test_p10_white_noise_scale():
    n, T, S = 256, 16, 40
    N = 2 * n
    h = si.hann_sinc_weights(n, T)
    rng = np.random.default_rng(11)
    sigma = 32.0
    L = N * (S + T - 1)
    s = sigma * rng.standard_normal((1, 1, L))
    Y = oracle.channelize_f64(s, n, T, h)["Y"][0, :, 1:, 0]
    expect = sigma ** 2 * np.sum(h.astype(np.float64) ** 2)
    assert abs(np.mean(np.abs(Y) ** 2) / expect - 1) < 0.05


# ------------------------------------------------------------------------------------------ P11
def test_p11_config1_channel100_prediction():
    (row,) = _golden_rows("config1_channel100.txt")
    mag, p0r, p0i, p1r, p1i = (float(v) for v in row.split())
    w = si.make_workload(1, sigma=0.0)                           # noise-free: tone only, rounded to integers
    res = oracle.process(w.packed, w.A, w.n, w.T, w.P, w.weights, w.S, coarse=w.coarse,
                         fine_delay=w.fine_delay, phase=w.phase, gains=w.gains)
    m = 64                                                       # steady state
    y0, y1 = res["Y"][0, m, 100, 0], res["Y"][0, m, 100, 1]
    assert abs(abs(y0) - mag) < 0.5 and abs(abs(y1) - mag) < 0.5
    assert abs(y0 - complex(p0r, p0i)) < 0.5
    assert abs(y1 - complex(p1r, p1i)) < 0.5
    np.testing.assert_array_equal(res["out"][0, m, 100, 0], [127, -127])      # both parts saturate
    assert res["out"][0, m, 100, 1, 0] == 127 and abs(int(res["out"][0, m, 100, 1, 1]) - 81) <= 1


# ------------------------------------------------------------------------------------------ P12
@pytest.mark.parametrize("n,T,S,per_spectrum", [(8, 1, 4, False), (16, 3, 6, False), (32, 4, 7, True), (64, 2, 5, True)])
def test_p12_whole_path_vs_definition(n, T, S, per_spectrum):
    w = si.custom_workload(A=2, n=n, T=T, S=S, seed=12, random_weights=True, per_spectrum=per_spectrum,
                           coarse_range=(-5, 2 * n + 9))
    for use_dft in (False, True):
        res = oracle.process(w.packed, w.A, w.n, w.T, w.P, w.weights, w.S, coarse=w.coarse,
                             fine_delay=w.fine_delay, phase=w.phase, gains=w.gains, use_dft=use_dft)
        for a in range(w.A):
            for p in range(w.P):
                for m in range(S):
                    mi = m if per_spectrum else 0
                    ref = brute_force(w.samples[a, p].astype(np.int64), n, T, w.weights, int(w.coarse[a, p, mi]),
                                      w.fine_delay[a, p, mi], w.phase[a, p, mi], w.gains[a, p], m)
                    got = res["Y"][a, m, :, p]
                    np.testing.assert_allclose(got, ref, rtol=0, atol=1e-9 * max(1.0, np.abs(ref).max()))
                    q = np.clip(np.rint(np.stack([ref.real, ref.imag], -1)), -127, 127)
                    near_tie = np.abs(np.abs(np.stack([ref.real, ref.imag], -1)) % 1 - 0.5) < 1e-6
                    assert np.all((res["out"][a, m, :, p] == q) | near_tie)


def test_direct_channel_agrees_with_fir_fft_route():
    w = si.custom_workload(A=1, n=64, T=4, S=6, seed=13, random_weights=True, per_spectrum=True,
                           coarse_range=(-3, 70))
    res = oracle.process(w.packed, 1, w.n, w.T, 2, w.weights, w.S, coarse=w.coarse, fine_delay=w.fine_delay,
                         phase=w.phase, gains=w.gains)
    rng = np.random.default_rng(0)
    for _ in range(20):
        p, m, k = int(rng.integers(2)), int(rng.integers(w.S)), int(rng.integers(w.n))
        y = oracle.direct_channel(w.packed[0, p], w.L, w.n, w.T, w.weights, m, int(w.coarse[0, p, m]),
                                  w.fine_delay[0, p, m], w.phase[0, p, m], w.gains[0, p, k], k)
        assert abs(y - res["Y"][0, m, k, p]) < 1e-9 * max(1.0, abs(y))


def test_selection_of_spectra_matches_full_run():
    w = si.custom_workload(A=2, n=32, T=4, S=12, seed=14, per_spectrum=True)
    full = oracle.process(w.packed, w.A, w.n, w.T, w.P, w.weights, w.S, coarse=w.coarse,
                          fine_delay=w.fine_delay, phase=w.phase, gains=w.gains)
    sel = np.array([0, 5, 11, 3])
    part = oracle.process(w.packed, w.A, w.n, w.T, w.P, w.weights, w.S, coarse=w.coarse,
                          fine_delay=w.fine_delay, phase=w.phase, gains=w.gains, sel=sel)
    np.testing.assert_array_equal(part["Y"], full["Y"][:, sel])
    np.testing.assert_array_equal(part["out"], full["out"][:, sel])


# ---------------------------------------------------------------------------------------------
# P1b  other sample widths (PAPER.md:273-279 bit-depth sweep): same bit-stream convention as R1
# ---------------------------------------------------------------------------------------------
def _pack_strings(values, bits):
    """Independent packer: binary strings, no shifts shared with oracle or generators."""
    stream = "".join(format(int(v) & ((1 << bits) - 1), f"0{bits}b") for v in values)
    assert len(stream) % 8 == 0
    return np.array([int(stream[i:i + 8], 2) for i in range(0, len(stream), 8)], dtype=np.uint8)


@pytest.mark.parametrize("bits", [4, 8, 10, 12, 16])
def test_unpack_bits_every_code_round_trips(bits):
    lo, hi = -(1 << (bits - 1)), (1 << (bits - 1)) - 1
    codes = np.arange(lo, hi + 1, dtype=np.int64)
    rng = np.random.default_rng(bits)
    codes = np.concatenate([codes, rng.integers(lo, hi + 1, size=64)])       # and a shuffled tail
    got = oracle.unpack_bits(_pack_strings(codes, bits), codes.size, bits)
    np.testing.assert_array_equal(got.astype(np.int64), codes)
    np.testing.assert_array_equal(si.pack_bits(codes, bits), _pack_strings(codes, bits))   # the generator's packer too


def test_unpack_bits_at_10_bits_is_unpack10_and_hand_examples():
    rng = np.random.default_rng(3)
    s = rng.integers(-512, 512, size=256)
    pk = si.pack10(s)
    np.testing.assert_array_equal(oracle.unpack_bits(pk, s.size, 10), oracle.unpack10(pk, s.size))
    # hand examples: 4-bit [1, -1, 7, -8] = 0x1F 0x78; 12-bit [1, -1] = 0x00 0x1F 0xFF; 16-bit [-2] = 0xFF 0xFE
    np.testing.assert_array_equal(oracle.unpack_bits(np.array([0x1F, 0x78], np.uint8), 4, 4), [1, -1, 7, -8])
    np.testing.assert_array_equal(oracle.unpack_bits(np.array([0x00, 0x1F, 0xFF], np.uint8), 2, 12), [1, -1])
    np.testing.assert_array_equal(oracle.unpack_bits(np.array([0xFF, 0xFE], np.uint8), 1, 16), [-2])


def test_one_lsb_in_one_sample_moves_every_channel_of_a_one_hot_spectrum():
    """The detection bound used by tests/test_gpu_parity.py::test_unpack_and_delay_are_exact_through_the_kernels_of_every_path:
    with weights = 1 at one tap, unit gain and no fine delay the spectrum is the transform of one integer row
    (PAPER.md:33-37), so one sample that is off by 1 LSB changes every channel by exactly 1 in modulus, i.e. by at least
    0.707 in its larger component -- far above that test's 0.3 bound."""
    n, T, S = 64, 4, 5
    N = 2 * n
    w = si.custom_workload(A=1, n=n, T=T, S=S, seed=3, sigma=8.0)
    j0 = 3
    h = np.zeros(N * T, dtype=np.float32)
    h[N * j0:N * (j0 + 1)] = 1.0
    c = np.array([[[5], [-9]]], dtype=np.int32)
    base = oracle.process(w.packed, 1, n, T, 2, h, S, coarse=c)["Y"]
    s = w.samples.copy()
    m, t = 2, 37
    u = N * (m + j0) - int(c[0, 1, 0]) + t                    # the sample row j0 of spectrum m reads at column t (pol 1)
    s[0, 1, u] += 1 if s[0, 1, u] < 511 else -1
    moved = oracle.process(si.pack10(s), 1, n, T, 2, h, S, coarse=c)["Y"]
    d = moved - base
    np.testing.assert_allclose(np.abs(d[0, m, :, 1]), 1.0, atol=1e-9)
    assert np.maximum(np.abs(d.real), np.abs(d.imag))[0, m, :, 1].min() >= 0.7
    d[0, m, :, 1] = 0
    assert np.abs(d).max() < 1e-9                             # and nothing else moves
