"""ctypes binding with the same names as include/fengine.h (argument marshalling only)."""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
_LIB_PATH = _PKG / "libfengine_b200.so"
_lib = None

# every symbol include/fengine.h declares (checked by tests/test_abi.py against the header text)
EXPORTED_SYMBOLS = [
    "fengine_create", "fengine_create_batched", "fengine_destroy", "fengine_set_coarse_delays",
    "fengine_set_fine_delays", "fengine_set_gains", "fengine_process", "fengine_process_host",
    "fengine_last_error", "fengine_process_f32", "fengine_debug_unpack", "fengine_debug_fir",
    "fengine_set_option", "fengine_last_launch_count", "fengine_profile_read", "fengine_process_heaps",
    "fengine_stream_begin", "fengine_stream_push", "fengine_stream_end", "fengine_reserve", "fengine_debug_pipe_stats", "fengine_debug_fp32_rate", "fengine_debug_path",
    "fengine_process_noalloc",
]

STATUS = {0: "OK", 1: "INVALID_ARG", 2: "ALLOC", 3: "CUDA", 4: "STATE"}


class FEngineError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"fengine error {code} ({STATUS.get(code, '?')}): {msg}")
        self.code = code


def library_path() -> Path:
    return _LIB_PATH


def lib() -> C.CDLL:
    """Load the CUDA library; fails loudly if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not _LIB_PATH.exists():
            raise FileNotFoundError(
                f"{_LIB_PATH} is missing: build it with `python -m paper_2303_09886_b200.build` "
                "(there is no CPU fallback)")
        L = C.CDLL(str(_LIB_PATH))
        vp, i64 = C.c_void_p, C.c_int64
        L.fengine_create.argtypes = [C.c_int, C.c_int, C.c_int, vp]
        L.fengine_create.restype = vp
        L.fengine_create_batched.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, vp]
        L.fengine_create_batched.restype = vp
        L.fengine_destroy.argtypes = [vp]
        L.fengine_destroy.restype = None
        L.fengine_set_coarse_delays.argtypes = [vp, vp, i64]
        L.fengine_set_fine_delays.argtypes = [vp, vp, vp, i64]
        L.fengine_set_gains.argtypes = [vp, vp]
        L.fengine_process.argtypes = [vp, vp, vp, i64, vp]
        L.fengine_process_host.argtypes = [vp, vp, vp, i64]
        L.fengine_reserve.argtypes = [vp, i64]
        L.fengine_debug_pipe_stats.argtypes = [vp, vp, i64]
        L.fengine_debug_fp32_rate.argtypes = [vp, vp]
        L.fengine_debug_path.argtypes = [vp]
        L.fengine_process_heaps.argtypes = [vp, vp, vp, i64, vp]
        L.fengine_stream_begin.argtypes = [vp, i64, vp]
        L.fengine_stream_push.argtypes = [vp, vp, vp, i64, vp]
        L.fengine_stream_end.argtypes = [vp]
        L.fengine_process_f32.argtypes = [vp, vp, vp, i64, vp]
        L.fengine_debug_unpack.argtypes = [vp, vp, vp, i64, vp]
        L.fengine_debug_fir.argtypes = [vp, vp, vp, i64, vp]
        L.fengine_last_error.argtypes = [vp]
        L.fengine_last_error.restype = C.c_char_p
        L.fengine_set_option.argtypes = [vp, C.c_char_p, i64]
        L.fengine_profile_read.argtypes = [vp, vp, vp, vp, vp]
        L.fengine_last_launch_count.argtypes = [vp]
        L.fengine_last_launch_count.restype = i64
        L.fengine_process_noalloc.argtypes = [vp, vp, vp, vp, vp, vp, vp, C.c_int, C.c_int, C.c_int, C.c_int, i64, vp,
                                              C.c_char_p, i64]
        _lib = L
    return _lib


def _host_ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _dev_ptr(t) -> int:
    """Device pointer of a torch CUDA tensor (or a raw int)."""
    if isinstance(t, int):
        return t
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    return t.data_ptr()


def _dev_buf(t, need_bytes: int, what: str, dtypes=None) -> int:
    """Device pointer of a contiguous CUDA tensor holding at least need_bytes (raw ints pass unchecked)."""
    if isinstance(t, int):
        return t
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError(f"{what}: expected a contiguous CUDA tensor")
    if dtypes is not None and str(t.dtype).replace("torch.", "") not in dtypes:
        raise ValueError(f"{what}: dtype {t.dtype}, expected one of {dtypes}")
    have = t.numel() * t.element_size()
    if have < need_bytes:
        raise ValueError(f"{what}: {have} bytes, the call needs {need_bytes}")
    return t.data_ptr()


def _stream_handle(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def fp32_rate() -> float:
    """fengine_debug_fp32_rate: sustained packed-FP32 rate of the current device in lane-operations per second."""
    r, ms = C.c_double(), C.c_double()
    rc = lib().fengine_debug_fp32_rate(C.byref(r), C.byref(ms))
    if rc != 0:
        raise FEngineError(rc, "fengine_debug_fp32_rate failed")
    return float(r.value)


NOALLOC_MAX_FLOATS = 1 << 20     # FENGINE_NOALLOC_MAX_FLOATS of include/fengine.h


def process_noalloc(inp, out, weights, coarse, fine_delay, phase, gains, n_antennas: int, n_channels: int, taps: int,
                    n_pols: int, n_spectra: int, stream=None):
    """fengine_process_noalloc: the whole path for callers that must not allocate device memory (a program that gave
    the GPU's memory to its own pool, a real-time loop that cannot stall on cudaMalloc).  No handle: every table is a
    CUDA tensor the caller already holds (weights float32 [N*T], coarse int32 [A][P], fine_delay / phase float32
    [A][P], gains float32 [A][P][n][2] or complex64 [A][P][n]); the intermediate lives in a 4 MiB array inside the
    library, which bounds A*P*n_spectra*N to NOALLOC_MAX_FLOATS and is shared by all calls (do not overlap them).
    Asynchronous on `stream`; make the first call on a device outside stream capture."""
    A, n, T, P, S = int(n_antennas), int(n_channels), int(taps), int(n_pols), int(n_spectra)
    N = 2 * n
    s_pos = max(S, 0)
    args = [
        _dev_buf(inp, A * P * (N * (s_pos + T - 1) * 10 // 8) if s_pos else 0, "input", ("uint8", "int8")),
        _dev_buf(out, A * s_pos * n * P * 2, "output", ("int8", "uint8")),
        _dev_buf(weights, N * T * 4, "weights", ("float32",)),
        _dev_buf(coarse, A * P * 4, "coarse", ("int32",)),
        _dev_buf(fine_delay, A * P * 4, "fine_delay", ("float32",)),
        _dev_buf(phase, A * P * 4, "phase", ("float32",)),
        _dev_buf(gains, A * P * n * 8, "gains", ("float32", "complex64")),
    ]
    err = C.create_string_buffer(512)
    rc = lib().fengine_process_noalloc(*args, A, n, T, P, S, _stream_handle(stream), err, len(err))
    if rc != 0:
        raise FEngineError(rc, err.value.decode())


class FEngine:
    """One engine: A antennas x P pols sharing the PFB weights (fengine_create_batched)."""

    def __init__(self, n_channels: int, taps: int, n_pols: int, weights, n_antennas: int = 1):
        w = np.ascontiguousarray(weights, dtype=np.float32).reshape(-1)
        if w.size != 2 * n_channels * taps:
            raise ValueError("weights must hold 2*n_channels*taps floats")
        self._lib = lib()
        self.A, self.n, self.T, self.P = n_antennas, n_channels, taps, n_pols
        self.N = 2 * n_channels
        self._h = self._lib.fengine_create_batched(n_antennas, n_channels, taps, n_pols, _host_ptr(w))
        if not self._h:
            raise FEngineError(3, "fengine_create_batched failed (invalid arguments, no CUDA device, or allocation)")

    # -- lifetime -----------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None):
            self._lib.fengine_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int):
        if rc != 0:
            raise FEngineError(rc, self._lib.fengine_last_error(self._h).decode())

    # -- setters (host arrays) ------------------------------------------------------------------
    def set_coarse_delays(self, c):
        c = np.ascontiguousarray(c, dtype=np.int32).reshape(self.A, self.P, -1)
        self._check(self._lib.fengine_set_coarse_delays(self._h, _host_ptr(c), c.shape[2]))

    def set_fine_delays(self, delay, phase):
        d = np.ascontiguousarray(delay, dtype=np.float32).reshape(self.A, self.P, -1)
        p = np.ascontiguousarray(phase, dtype=np.float32).reshape(self.A, self.P, -1)
        if d.shape != p.shape:
            raise ValueError("delay and phase must have the same shape")
        self._check(self._lib.fengine_set_fine_delays(self._h, _host_ptr(d), _host_ptr(p), d.shape[2]))

    def set_gains(self, gains):
        g = np.ascontiguousarray(np.asarray(gains, dtype=np.complex64).reshape(self.A, self.P, self.n))
        self._check(self._lib.fengine_set_gains(self._h, _host_ptr(g.view(np.float32))))

    def set_option(self, key: str, value: int):
        self._check(self._lib.fengine_set_option(self._h, key.encode(), int(value)))
        if key == "sample_bits":
            self.sample_bits = int(value)

    # -- sizes ----------------------------------------------------------------------------------
    def input_bytes(self, n_spectra: int) -> int:
        return self.A * self.P * (self.N * (n_spectra + self.T - 1) * getattr(self, "sample_bits", 10) // 8)

    def output_shape(self, n_spectra: int):
        return (self.A, n_spectra, self.n, self.P, 2)

    def reserve(self, max_spectra: int):
        """fengine_reserve: size every buffer now so that process() never allocates."""
        self._check(self._lib.fengine_reserve(self._h, int(max_spectra)))

    def _in(self, t, n_spectra: int) -> int:
        return _dev_buf(t, self.input_bytes(max(n_spectra, 0)) if n_spectra > 0 else 0, "input", ("uint8", "int8"))

    def _out(self, t, n_spectra: int, itemsize: int = 1, dtypes=("int8", "uint8")) -> int:
        need = int(np.prod(self.output_shape(max(n_spectra, 0)))) * itemsize
        return _dev_buf(t, need, "output", dtypes)

    # -- the hot path -----------------------------------------------------------------------------
    def process(self, inp, out, n_spectra: int, stream=None):
        """fengine_process: device tensors (uint8 in, int8 out); asynchronous on `stream`."""
        self._check(self._lib.fengine_process(self._h, self._in(inp, n_spectra), self._out(out, n_spectra), n_spectra,
                                              _stream_handle(stream)))

    def heaps_shape(self, n_spectra: int):
        return (self.A, (n_spectra + 255) // 256, self.n, 256, self.P, 2)

    def process_heaps(self, inp, heaps_out, n_spectra: int, stream=None):
        """fengine_process_heaps: channel-major heaps of 256 spectra (int8, shape heaps_shape(n_spectra))."""
        need = int(np.prod(self.heaps_shape(max(n_spectra, 0))))
        self._check(self._lib.fengine_process_heaps(self._h, self._in(inp, n_spectra),
                                                    _dev_buf(heaps_out, need, "heaps", ("int8", "uint8")), n_spectra,
                                                    _stream_handle(stream)))

    def stream_begin(self, max_new_spectra: int) -> int:
        """fengine_stream_begin; returns the latency D in spectra."""
        d = C.c_int64(0)
        self._check(self._lib.fengine_stream_begin(self._h, max_new_spectra, C.byref(d)))
        return int(d.value)

    def stream_push(self, inp_new, out, n_new: int, stream=None):
        row_bytes = self.N * getattr(self, "sample_bits", 10) // 8
        need_in = self.A * self.P * max(n_new, 0) * row_bytes                  # the new rows only: the library keeps history
        self._check(self._lib.fengine_stream_push(self._h, _dev_buf(inp_new, need_in, "input", ("uint8", "int8")),
                                                  self._out(out, n_new), n_new, _stream_handle(stream)))

    def stream_end(self):
        self._check(self._lib.fengine_stream_end(self._h))

    def process_f32(self, inp, out_f32, n_spectra: int, stream=None):
        self._check(self._lib.fengine_process_f32(self._h, self._in(inp, n_spectra),
                                                  self._out(out_f32, n_spectra, 4, ("float32",)), n_spectra,
                                                  _stream_handle(stream)))

    def process_host(self, inp_host, out_host, n_spectra: int):
        """fengine_process_host: host buffers (numpy or pinned torch tensors); synchronous."""
        def hp(x, need, what):
            if isinstance(x, np.ndarray):
                if not x.flags["C_CONTIGUOUS"] or x.nbytes < need:
                    raise ValueError(f"{what}: expected a C-contiguous array of at least {need} bytes")
                return x.ctypes.data
            if x.is_cuda or not x.is_contiguous() or x.numel() * x.element_size() < need:
                raise ValueError(f"{what}: expected a contiguous host tensor of at least {need} bytes")
            return x.data_ptr()
        n_out = int(np.prod(self.output_shape(max(n_spectra, 0))))
        self._check(self._lib.fengine_process_host(self._h, hp(inp_host, self.input_bytes(n_spectra) if n_spectra > 0 else 0, "input"),
                                                   hp(out_host, n_out, "output"), n_spectra))

    def debug_unpack(self, inp, out_i16, n_spectra: int, stream=None):
        need = self.A * self.P * max(n_spectra, 0) * self.N * self.T * 2
        self._check(self._lib.fengine_debug_unpack(self._h, self._in(inp, n_spectra), _dev_buf(out_i16, need, "samples", ("int16",)),
                                                   n_spectra, _stream_handle(stream)))

    def debug_fir(self, inp, out_f32, n_spectra: int, stream=None):
        need = self.A * self.P * max(n_spectra, 0) * self.N * 4
        self._check(self._lib.fengine_debug_fir(self._h, self._in(inp, n_spectra), _dev_buf(out_f32, need, "g", ("float32",)),
                                                n_spectra, _stream_handle(stream)))

    def profile_read(self):
        """(fir_ms, fft_ms, n_fir, n_fft) summed since the last read (option "profile" must be 1)."""
        a, b = C.c_double(), C.c_double()
        na, nb = C.c_int64(), C.c_int64()
        self._check(self._lib.fengine_profile_read(self._h, C.byref(a), C.byref(b), C.byref(na), C.byref(nb)))
        return a.value, b.value, na.value, nb.value

    def pipe_stats(self, n_sms: int = 148):
        """fengine_debug_pipe_stats: [n_sms][16] uint64 clock counters of the pipelined kernel (option pipe_stats)."""
        out = np.zeros((n_sms, 16), dtype=np.uint64)
        self._check(self._lib.fengine_debug_pipe_stats(self._h, _host_ptr(out), out.size))
        return out

    PATHS = {0: "generic", 1: "one_pol", 2: "pol_packed", 3: "packed_fir_one_pol_fft", 4: "fused", 5: "split"}

    def path(self) -> str:
        """fengine_debug_path: which kernels process() would launch now."""
        return self.PATHS[int(self._lib.fengine_debug_path(self._h))]

    def last_launch_count(self) -> int:
        return int(self._lib.fengine_last_launch_count(self._h))
