"""Seeded synthetic inputs for the F-engine path (serves the tests, bench.py and smoke()).

This module holds NONE of the method's arithmetic: it only *produces* inputs --
10-bit samples packed into bytes, filter weights, delay tables, gains -- with the
shapes and distributions of the paper's workloads (PAPER.md:31, :39, :51, :227,
:315; BASELINE.json configs).  It stands in for the MeerKAT digitiser streams,
which are not available; the recipe is stated in DESIGN.md ("Input recipe").

Neither oracle/ nor paper_2303_09886_b200/ is imported here.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

__all__ = ["pack10", "pack_bits", "pack10_bitwise", "hann_sinc_weights", "Workload", "make_workload", "custom_workload",
           "CONFIG_SHAPES"]


# ---------------------------------------------------------------------------------------------
# 10-bit packing (4096 samples in 5120 bytes; bit order per BASELINE.json configs[0]:
# two's complement, MSB first, 4 samples per 5 bytes).  Written as a generic bit-stream writer
# (a 16-bit window per sample) so that it does not mirror the unpack formula of either side.
# ---------------------------------------------------------------------------------------------
def pack10(samples: np.ndarray) -> np.ndarray:
    """Pack int samples in [-512, 511] (last axis, length % 4 == 0) into bytes (length * 5 / 4)."""
    s = np.asarray(samples)
    assert s.shape[-1] % 4 == 0
    assert s.min(initial=0) >= -512 and s.max(initial=0) <= 511
    lead = s.shape[:-1]
    L = s.shape[-1]
    v = (s.astype(np.int32) & 0x3FF).astype(np.uint16).reshape(-1, L // 4, 4)
    out = np.zeros((v.shape[0], L // 4, 5), dtype=np.uint8)
    for r in range(4):
        bitpos = 10 * r                       # within the 40-bit group
        byte0, off = bitpos >> 3, bitpos & 7
        w = (v[:, :, r].astype(np.uint32) << (6 - off)).astype(np.uint16)   # 10 bits inside a 16-bit window
        out[:, :, byte0] |= (w >> 8).astype(np.uint8)
        out[:, :, byte0 + 1] |= (w & 0xFF).astype(np.uint8)
    return out.reshape(*lead, L // 4 * 5)


def pack_bits(samples: np.ndarray, bits: int) -> np.ndarray:
    """Pack int samples (last axis) as `bits`-bit two's complement, MSB first (the convention of pack10; the
    bit-depth sweep of PAPER.md:273-279 uses 4, 8, 12 and 16 bits).  length * bits must be a multiple of 8."""
    s = np.asarray(samples)
    L = s.shape[-1]
    assert 1 <= bits <= 16 and (L * bits) % 8 == 0
    assert s.min(initial=0) >= -(1 << (bits - 1)) and s.max(initial=0) <= (1 << (bits - 1)) - 1
    if bits == 10:
        return pack10(s)
    lead = s.shape[:-1]
    v = (s.astype(np.int32) & ((1 << bits) - 1)).astype(np.uint32).reshape(-1, L)
    if bits == 8:
        out = v.astype(np.uint8)
    elif bits == 16:
        out = np.stack([(v >> 8).astype(np.uint8), (v & 0xFF).astype(np.uint8)], axis=-1).reshape(v.shape[0], -1)
    elif bits == 4:
        out = ((v[:, 0::2] << 4) | v[:, 1::2]).astype(np.uint8)
    elif bits == 12:
        a, b = v[:, 0::2], v[:, 1::2]
        out = np.stack([(a >> 4).astype(np.uint8), (((a & 15) << 4) | (b >> 8)).astype(np.uint8),
                        (b & 0xFF).astype(np.uint8)], axis=-1).reshape(v.shape[0], -1)
    else:
        bitsarr = ((v[:, :, None] >> np.arange(bits - 1, -1, -1)) & 1).astype(np.uint8).reshape(v.shape[0], -1)
        out = np.packbits(bitsarr, axis=-1)
    return out.reshape(*lead, L * bits // 8)


def pack10_bitwise(samples) -> np.ndarray:
    """Slow bit-by-bit packer (pure Python) used to pin both pack10 and the unpackers."""
    bits = []
    for s in samples:
        v = int(s) & 0x3FF
        for b in range(9, -1, -1):
            bits.append((v >> b) & 1)
    assert len(bits) % 8 == 0
    out = np.zeros(len(bits) // 8, dtype=np.uint8)
    for i, bit in enumerate(bits):
        out[i >> 3] |= bit << (7 - (i & 7))
    return out


# ---------------------------------------------------------------------------------------------
# PFB weights: Hann-windowed sinc, formula per BASELINE.json configs[0] and R14:
#   h[m] = sinc((m - T n) / (2n)) * hann(m),  hann(m) = 0.5 - 0.5 cos(2 pi m / (2 n T)),  m < 2nT
# The weights are an INPUT of the path (fengine_create takes them), so this is a generator.
# ---------------------------------------------------------------------------------------------
def hann_sinc_weights(n: int, T: int) -> np.ndarray:
    N = 2 * n
    m = np.arange(N * T, dtype=np.float64)
    h = np.sinc((m - T * n) / N) * (0.5 - 0.5 * np.cos(2.0 * np.pi * m / (N * T)))
    return h.astype(np.float32)


# (A, n, T, L-per-stream) of BASELINE.json configs 1..5 (config 5 listed at n = 4096; others via n=)
CONFIG_SHAPES = {
    1: dict(A=1, n=1024, T=16, S=128),
    2: dict(A=4, n=4096, T=16, L=1 << 24),
    3: dict(A=4, n=32768, T=16, L=1 << 26),
    4: dict(A=8, n=8192, T=16, L=1 << 25),
    5: dict(A=16, n=4096, T=16, L=1 << 26),
}


@dataclass
class Workload:
    name: str
    A: int
    P: int
    n: int
    T: int
    S: int                                   # spectra per call
    packed: np.ndarray                       # uint8 [A][P][L*5/4]
    weights: np.ndarray                      # float32 [N*T]
    coarse: np.ndarray                       # int32 [A][P][1 or S]
    fine_delay: np.ndarray                   # float32 [A][P][1 or S]
    phase: np.ndarray                        # float32 [A][P][1 or S]
    gains: np.ndarray                        # complex64 [A][P][n]
    samples: np.ndarray | None = None        # int16 [A][P][L] (kept on request)
    meta: dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return 2 * self.n

    @property
    def L(self) -> int:
        return self.N * (self.S + self.T - 1)


def _samples(rng, L, N, sigma, tones, bits: int = 10):
    """clip(rint(sigma * N(0,1) + sum A_i cos(2 pi k_i u / N + theta_i)), -2^(b-1), 2^(b-1) - 1); tones are on-bin."""
    x = rng.standard_normal(L, dtype=np.float32)
    x *= np.float32(sigma)
    if tones:
        u = np.arange(N, dtype=np.float64)
        period = np.zeros(N, dtype=np.float64)
        for (k, amp, theta) in tones:
            period += amp * np.cos(2.0 * np.pi * ((k * u) % N) / N + theta)
        reps = -(-L // N)
        x += np.tile(period.astype(np.float32), reps)[:L]
    np.rint(x, out=x)
    np.clip(x, -(1 << (bits - 1)), (1 << (bits - 1)) - 1, out=x)
    return x.astype(np.int16)


def _random_gains(prng, A, P, n):
    mag = 0.01 * (1.0 + 0.1 * prng.standard_normal((A, P, n)))
    ang = 2.0 * np.pi * prng.random((A, P, n))
    return (mag * np.exp(1j * ang)).astype(np.complex64)


def make_workload(config: int, n_spectra: int | None = None, n_antennas: int | None = None,
                  n_channels: int | None = None, seed: int = 0, keep_samples: bool = False,
                  sigma: float | None = None, taps: int | None = None, bits: int = 10) -> Workload:
    """Build the synthetic stand-in for BASELINE.json config `config` (1..5).

    n_spectra / n_antennas shrink the batch (same distributions) so that the oracle finishes in
    seconds; n_channels selects the sweep point of config 5.  `sigma` overrides the noise level
    (config 4 variant 4b uses sigma=182, R17).  `taps` overrides T (the paper's tap sweep); `bits` != 10 packs
    the samples at another width (bit-depth sweep) with sigma and tone amplitudes scaled by
    2^(bits - 10), so that the signal fills the range the same way.
    """
    shp = dict(CONFIG_SHAPES[config])
    A = n_antennas or shp["A"]
    n = n_channels or shp["n"]
    T = taps or shp["T"]
    P = 2
    N = 2 * n
    if n_spectra is None:
        n_spectra = shp["S"] if "S" in shp else shp["L"] // N - (T - 1)
    S = int(n_spectra)
    L = N * (S + T - 1)
    prng = np.random.default_rng([seed, config, 10 ** 6])      # per-engine parameters
    weights = hann_sinc_weights(n, T)

    if config == 1:
        sig = 32.0 if sigma is None else sigma
        tones = [[(100 % n, 64.0, 0.0)] for _ in range(A)]
        coarse = np.tile(np.array([3, 0], dtype=np.int32).reshape(1, 2, 1), (A, 1, 1))
        fine = np.full((A, P, 1), 0.25, dtype=np.float32)
        phase = np.full((A, P, 1), 0.1, dtype=np.float32)
        gains = np.full((A, P, n), 0.01 * (1 + 0.1j), dtype=np.complex64)
    elif config in (2, 3, 5):
        sig = 32.0 if sigma is None else sigma
        if config == 2:
            tones = [[(int(prng.integers(1, n)), 64.0, float(2 * np.pi * prng.random()))] for _ in range(A)]
        elif config == 3:
            tones = [[(int(prng.integers(1, n)), 32.0, float(2 * np.pi * prng.random())) for _ in range(5)]
                     for _ in range(A)]
        else:
            tones = [[] for _ in range(A)]
        c = prng.integers(0, N if config != 2 else 4096, size=A).astype(np.int32)
        coarse = np.repeat(c.reshape(A, 1, 1), P, axis=1)
        d = prng.uniform(-0.5, 0.5, size=A).astype(np.float32)
        ph = prng.uniform(0.0, 2 * np.pi, size=A).astype(np.float32)
        fine = np.repeat(d.reshape(A, 1, 1), P, axis=1)
        phase = np.repeat(ph.reshape(A, 1, 1), P, axis=1)
        gains = _random_gains(prng, A, P, n)
    elif config == 4:
        sig = 100.0 if sigma is None else sigma
        tones = [[] for _ in range(A)]
        c0 = prng.integers(0, N, size=A).astype(np.int64)
        m = np.arange(S, dtype=np.int64)
        c = (c0[:, None] + m[None, :] // 64).astype(np.int32)                    # +1 sample every 64 spectra
        coarse = np.repeat(c.reshape(A, 1, S), P, axis=1)
        d0 = prng.uniform(-0.5, 0.5, size=A)
        d = (d0[:, None] + 1e-3 * m[None, :]).astype(np.float32)                 # ramps 1e-3 samples / spectrum
        fine = np.repeat(d.reshape(A, 1, S), P, axis=1)
        ph = prng.uniform(0.0, 2 * np.pi, size=A).astype(np.float32)
        phase = np.repeat(np.repeat(ph.reshape(A, 1, 1), P, axis=1), S, axis=2)
        gains = _random_gains(prng, A, P, n)
    else:
        raise ValueError(config)

    scale = 2.0 ** (bits - 10)
    packed = np.empty((A, P, L * bits // 8), dtype=np.uint8)
    samples = np.empty((A, P, L), dtype=np.int16) if keep_samples else None
    def one_stream(ap):
        a, p = ap
        rng = np.random.default_rng([seed, config, a, p])       # one generator per stream: the result does not depend
        tn = tones[a] if bits == 10 else [(k, amp * scale, th) for (k, amp, th) in tones[a]]      # on the thread count
        s = _samples(rng, L, N, sig * scale, tn, bits)          # tone common to both pols, independent noise
        packed[a, p] = pack_bits(s, bits)
        if keep_samples:
            samples[a, p] = s

    streams = [(a, p) for a in range(A) for p in range(P)]
    if L * len(streams) >= 1 << 24:                             # large batches: numpy releases the GIL in these loops
        from concurrent.futures import ThreadPoolExecutor
        import os
        with ThreadPoolExecutor(max_workers=min(len(streams), os.cpu_count() or 1)) as ex:
            list(ex.map(one_stream, streams))
    else:
        for ap in streams:
            one_stream(ap)
    return Workload(name=f"config{config}", A=A, P=P, n=n, T=T, S=S, packed=packed, weights=weights,
                    coarse=np.ascontiguousarray(coarse), fine_delay=np.ascontiguousarray(fine),
                    phase=np.ascontiguousarray(phase), gains=gains, samples=samples,
                    meta=dict(config=config, sigma=sig, tones=tones, seed=seed, bits=bits))


def custom_workload(A: int, n: int, T: int, S: int, P: int = 2, seed: int = 0, sigma: float = 32.0,
                    coarse_range: tuple[int, int] | None = None, per_spectrum: bool = False,
                    random_weights: bool = False, keep_samples: bool = True, tag: int = 99, bits: int = 10) -> Workload:
    """Small free-form workload for edge-case parity tests (tiny n, odd T, negative delays, ...).  `bits` != 10
    packs the samples at another depth (sigma is the caller's business; the range is clipped to `bits`)."""
    N = 2 * n
    L = N * (S + T - 1)
    prng = np.random.default_rng([seed, tag, 10 ** 6, A, n, T, S])
    if random_weights:
        weights = prng.standard_normal(N * T).astype(np.float32)          # asymmetric: pins tap order (R5)
    else:
        weights = hann_sinc_weights(n, T)
    lo, hi = coarse_range if coarse_range is not None else (0, N)
    nper = S if per_spectrum else 1
    coarse = prng.integers(lo, hi, size=(A, P, nper)).astype(np.int32)
    fine = prng.uniform(-0.5, 0.5, size=(A, P, nper)).astype(np.float32)
    phase = prng.uniform(0, 2 * np.pi, size=(A, P, nper)).astype(np.float32)
    gains = _random_gains(prng, A, P, n)
    packed = np.empty((A, P, L * bits // 8), dtype=np.uint8)
    samples = np.empty((A, P, L), dtype=np.int16) if keep_samples else None
    for a in range(A):
        for p in range(P):
            rng = np.random.default_rng([seed, tag, a, p, n, S])
            k = int(rng.integers(1, max(n, 2)))
            s = _samples(rng, L, N, sigma, [(k, 2 * sigma, float(rng.random()))], bits)
            packed[a, p] = pack_bits(s, bits)
            if keep_samples:
                samples[a, p] = s
    return Workload(name=f"custom_A{A}_n{n}_T{T}_S{S}", A=A, P=P, n=n, T=T, S=S, packed=packed,
                    weights=weights, coarse=coarse, fine_delay=fine, phase=phase, gains=gains,
                    samples=samples, meta=dict(seed=seed, sigma=sigma, bits=bits))
