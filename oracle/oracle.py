"""ctypes binding of oracle/fengine_oracle.c (argument marshalling only).

TEST INFRASTRUCTURE, NOT THE PRODUCT -- see fengine_oracle.c for the citations
(PAPER.md line numbers) of every function wrapped here.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "fengine_oracle.c"
_SO = _HERE / "libfengine_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not _SO.exists() or _SO.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _SO.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC", str(_SRC), "-o", str(tmp), "-lm"]
        )
        os.replace(tmp, _SO)
    return _SO


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_SO))
        p = C.c_void_p
        i64 = C.c_int64
        L.oracle_unpack10.argtypes = [p, i64, p]
        L.oracle_unpack10.restype = None
        L.oracle_window.argtypes = [p, i64, C.c_int, C.c_int, i64, i64, p]
        L.oracle_window.restype = None
        L.oracle_fir.argtypes = [p, p, C.c_int, C.c_int, p]
        L.oracle_fir.restype = None
        L.oracle_twiddles.argtypes = [C.c_int, p, p]
        L.oracle_twiddles.restype = None
        L.oracle_fft_radix2.argtypes = [p, p, C.c_int, p, p]
        L.oracle_fft_radix2.restype = None
        L.oracle_dft.argtypes = [p, C.c_int, C.c_int, p, p]
        L.oracle_dft.restype = None
        L.oracle_quantize.argtypes = [C.c_double]
        L.oracle_quantize.restype = C.c_int
        common = [C.c_int, C.c_int, C.c_int, C.c_int, p, p, i64, p, p, i64, p]
        L.oracle_channelize_f64.argtypes = common + [p, i64, p, i64, p, p, p, C.c_int, C.c_int]
        L.oracle_channelize_f64.restype = C.c_int
        L.oracle_process.argtypes = common + [p, i64, p, i64, p, p, p, C.c_int, C.c_int]
        L.oracle_process.restype = C.c_int
        L.oracle_direct_channel.argtypes = [p, i64, C.c_int, C.c_int, p, i64, i64, C.c_double, C.c_double,
                                            C.c_double, C.c_double, C.c_int, p, p]
        L.oracle_direct_channel.restype = None
        L.oracle_num_threads.argtypes = []
        L.oracle_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def unpack10(packed: np.ndarray, n_samples: int) -> np.ndarray:
    packed = np.ascontiguousarray(packed, dtype=np.uint8)
    assert packed.size >= (n_samples + 3) // 4 * 5
    out = np.empty(n_samples, dtype=np.int16)
    lib().oracle_unpack10(_ptr(packed), n_samples, _ptr(out))
    return out


def unpack_bits(packed: np.ndarray, n_samples: int, bits: int) -> np.ndarray:
    """b-bit two's complement samples, MSB first (PAPER.md:273-279 bit-depth sweep; convention of R1)."""
    packed = np.ascontiguousarray(packed, dtype=np.uint8)
    assert 1 <= bits <= 16 and packed.size * 8 >= n_samples * bits
    out = np.empty(n_samples, dtype=np.int16)
    L = lib()
    L.oracle_unpack_bits.argtypes = [C.c_void_p, C.c_int64, C.c_int, C.c_void_p]
    L.oracle_unpack_bits.restype = None
    L.oracle_unpack_bits(_ptr(packed), n_samples, bits, _ptr(out))
    return out


def window(s: np.ndarray, N: int, T: int, m: int, c: int) -> np.ndarray:
    s = np.ascontiguousarray(s, dtype=np.float64)
    x = np.empty(N * T, dtype=np.float64)
    lib().oracle_window(_ptr(s), s.size, N, T, m, c, _ptr(x))
    return x


def fir(x: np.ndarray, h: np.ndarray, N: int, T: int) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float64)
    h = np.ascontiguousarray(h, dtype=np.float32)
    assert x.size == N * T and h.size == N * T
    g = np.empty(N, dtype=np.float64)
    lib().oracle_fir(_ptr(x), _ptr(h), N, T, _ptr(g))
    return g


def fft_radix2(z: np.ndarray) -> np.ndarray:
    z = np.asarray(z, dtype=np.complex128)
    N = z.size
    re = np.ascontiguousarray(z.real)
    im = np.ascontiguousarray(z.imag)
    twr = np.empty(max(N // 2, 1), dtype=np.float64)
    twi = np.empty(max(N // 2, 1), dtype=np.float64)
    lib().oracle_twiddles(N, _ptr(twr), _ptr(twi))
    lib().oracle_fft_radix2(_ptr(re), _ptr(im), N, _ptr(twr), _ptr(twi))
    return re + 1j * im


def dft(g: np.ndarray, n_out: int | None = None) -> np.ndarray:
    g = np.ascontiguousarray(g, dtype=np.float64)
    N = g.size
    n_out = N if n_out is None else n_out
    re = np.empty(n_out, dtype=np.float64)
    im = np.empty(n_out, dtype=np.float64)
    lib().oracle_dft(_ptr(g), N, n_out, _ptr(re), _ptr(im))
    return re + 1j * im


def quantize(v: float) -> int:
    return int(lib().oracle_quantize(float(v)))


def _params(A, n, T, P, weights, coarse, fine_delay, phase, gains):
    N = 2 * n
    h = np.ascontiguousarray(weights, dtype=np.float32).reshape(-1)
    assert h.size == N * T, "weights must hold N*T floats, weights[t + N*j] = w[t][j]"
    if coarse is None:
        coarse = np.zeros((A, P, 1), dtype=np.int32)
    coarse = np.ascontiguousarray(coarse, dtype=np.int32).reshape(A, P, -1)
    if fine_delay is None:
        fine_delay = np.zeros((A, P, 1), dtype=np.float32)
    if phase is None:
        phase = np.zeros((A, P, 1), dtype=np.float32)
    fine_delay = np.ascontiguousarray(fine_delay, dtype=np.float32).reshape(A, P, -1)
    phase = np.ascontiguousarray(phase, dtype=np.float32).reshape(A, P, -1)
    assert fine_delay.shape == phase.shape
    if gains is None:
        gains = np.ones((A, P, n), dtype=np.complex64)
    gains = np.ascontiguousarray(np.asarray(gains, dtype=np.complex64).reshape(A, P, n))
    return h, coarse, fine_delay, phase, gains


def _run(fn, A, n, T, P, h, coarse, fd, ph, gains, data, length_arg, sel, n_sel, want_Y, want_nyq,
         use_dft, threads):
    if sel is not None:
        sel = np.ascontiguousarray(sel, dtype=np.int64)
        n_sel = sel.size
    out = np.empty((A, n_sel, n, P, 2), dtype=np.int8)
    Y = np.empty((A, n_sel, n, P, 2), dtype=np.float64) if want_Y else None
    nyq = np.empty((A, P, n_sel, 2), dtype=np.float64) if want_nyq else None
    if coarse.shape[2] != 1:
        need = (int(sel.max()) + 1) if sel is not None and sel.size else n_sel
        assert coarse.shape[2] >= need
    rc = fn(A, n, T, P, _ptr(h), _ptr(coarse), coarse.shape[2], _ptr(fd), _ptr(ph), fd.shape[2],
            _ptr(gains.view(np.float32)), _ptr(data), length_arg, _ptr(sel), n_sel,
            _ptr(out), _ptr(Y), _ptr(nyq), int(use_dft), int(threads))
    if rc != 0:
        raise RuntimeError(f"oracle returned {rc}")
    res = {"out": out}
    if want_Y:
        res["Y"] = Y[..., 0] + 1j * Y[..., 1]          # [A][S][n][P] complex128
    if want_nyq:
        res["nyquist"] = nyq[..., 0] + 1j * nyq[..., 1]  # [A][P][S]
    return res


def channelize_f64(samples, n, T, weights, coarse=None, fine_delay=None, phase=None, gains=None,
                   n_spectra=None, sel=None, want_Y=True, want_nyq=False, use_dft=False, threads=0):
    """Whole path on float64 samples [A][P][L] (no unpack step)."""
    s = np.ascontiguousarray(samples, dtype=np.float64)
    A, P, L = s.shape
    h, coarse, fd, ph, gains = _params(A, n, T, P, weights, coarse, fine_delay, phase, gains)
    if n_spectra is None:
        n_spectra = L // (2 * n) - (T - 1)
    return _run(lib().oracle_channelize_f64, A, n, T, P, h, coarse, fd, ph, gains, s, L, sel, n_spectra,
                want_Y, want_nyq, use_dft, threads)


def process(packed, A, n, T, P, weights, n_spectra, coarse=None, fine_delay=None, phase=None, gains=None,
            sel=None, want_Y=True, want_nyq=False, use_dft=False, threads=0):
    """Whole path on packed 10-bit input [A][P][L*5/4] bytes, L = 2n(n_spectra + T - 1)."""
    packed = np.ascontiguousarray(packed, dtype=np.uint8).reshape(-1)
    L = 2 * n * (n_spectra + T - 1)
    assert packed.size == A * P * (L // 4 * 5), (packed.size, A * P * (L // 4 * 5))
    h, coarse, fd, ph, gains = _params(A, n, T, P, weights, coarse, fine_delay, phase, gains)
    return _run(lib().oracle_process, A, n, T, P, h, coarse, fd, ph, gains, packed, n_spectra, sel, n_spectra,
                want_Y, want_nyq, use_dft, threads)


def direct_channel(stream_bytes, L, n, T, weights, m, c, d, phi, gain, k) -> complex:
    """The definition for one output value: NT-term windowed DTFT, then rotation and gain."""
    b = np.ascontiguousarray(stream_bytes, dtype=np.uint8)
    h = np.ascontiguousarray(weights, dtype=np.float32).reshape(-1)
    yr = C.c_double()
    yi = C.c_double()
    g = complex(gain)
    lib().oracle_direct_channel(_ptr(b), L, n, T, _ptr(h), m, c, float(np.float32(d)), float(np.float32(phi)),
                                float(np.float32(g.real)), float(np.float32(g.imag)), k,
                                C.byref(yr), C.byref(yi))
    return complex(yr.value, yi.value)
