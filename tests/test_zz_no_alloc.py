"""fengine_process_noalloc, the entry point for callers that must not allocate device memory.

Some users of the library cannot call cudaMalloc once they are running: an application that handed the whole GPU to
its own memory pool at start-up, or a real-time receive loop that cannot afford the device-wide stall
an allocation causes.  fengine_process_noalloc serves them: no handle, every table a device pointer the caller owns,
and the FIR -> transform intermediate in a fixed 4 MiB array built into the library (include/fengine.h).

This file checks that entry point against the existing path (an FEngine handle, which allocates) on the same inputs,
at the tolerance of tests/test_gpu_parity.py, on two calls in a row: all calls share the built-in array, which still
holds the first call's rows when the second one (a different shape and data) runs.  The file is named so that pytest
collects it last: `pytest -x` stops at the first failure, and a failure here must not hide the parity tests.  It makes
no assumption on what ran before it (it passes alone in a fresh process, where its first call does the per-device
set-up, and after the other tests).
"""
import numpy as np
import pytest

import synth_inputs as si

pytestmark = pytest.mark.gpu

INT8_MISMATCH = 1e-4    # fraction of int8 values allowed to differ by exactly 1 LSB (the bar of test_gpu_parity.py)


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def fb():
    import paper_2303_09886_b200 as fb
    fb.lib()            # fails loudly if the CUDA library is missing
    return fb


def _existing_path(torch, fb, w, **opts):
    """int8 output of fengine_process on a handle (the path that allocates its tables and scratch)."""
    fe = fb.FEngine(w.n, w.T, w.P, w.weights, n_antennas=w.A)
    fe.set_coarse_delays(w.coarse)
    fe.set_fine_delays(w.fine_delay, w.phase)
    fe.set_gains(w.gains)
    for k, v in opts.items():
        fe.set_option(k, v)
    d_in = torch.from_numpy(w.packed.reshape(-1)).cuda()
    d_out = torch.full(fe.output_shape(w.S), 99, dtype=torch.int8, device="cuda")
    fe.process(d_in, d_out, w.S)
    torch.cuda.synchronize()
    path = fe.path()
    fe.close()
    return d_out.cpu().numpy(), path


_kept = {}


def _no_alloc(torch, fb, w, keep=False):
    """int8 output of fengine_process_noalloc; the caller's buffers are made here, before the call (keep: reuse the
    buffers of the previous call for this workload, so that this function allocates nothing itself)."""
    dev = _kept.get(w.name) if keep else None
    if dev is not None:
        dev["out"].fill_(99)
    else:
        dev = _kept[w.name] = {
            "in": torch.from_numpy(w.packed.reshape(-1)).cuda(),
            "w": torch.from_numpy(w.weights).cuda(),
            "c": torch.from_numpy(np.ascontiguousarray(w.coarse[:, :, 0])).cuda(),
            "d": torch.from_numpy(np.ascontiguousarray(w.fine_delay[:, :, 0])).cuda(),
            "phi": torch.from_numpy(np.ascontiguousarray(w.phase[:, :, 0])).cuda(),
            "g": torch.from_numpy(np.ascontiguousarray(w.gains).view(np.float32)).cuda(),
            "out": torch.full((w.A, w.S, w.n, w.P, 2), 99, dtype=torch.int8, device="cuda"),
        }
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    fb.process_noalloc(dev["in"], dev["out"], dev["w"], dev["c"], dev["d"], dev["phi"], dev["g"], w.A, w.n, w.T, w.P, w.S)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before      # nothing went through torch's allocator either
    return dev["out"].cpu().numpy()


def _assert_same(got, want, label):
    g, r = got.astype(np.int32), want.astype(np.int32)
    assert g.shape == r.shape
    d = np.abs(g - r)
    assert d.max() <= 1, f"{label}: int8 differs by more than 1 LSB (max {d.max()})"
    frac = np.count_nonzero(d) / d.size
    assert frac <= INT8_MISMATCH, f"{label}: {frac:.2e} of int8 values differ"
    assert g.min() >= -127 and g.max() <= 127


def test_no_alloc_entry_point_matches_the_existing_path_on_two_calls_in_a_row(torch, fb):
    # call 1: config 1 (n = 1024, 16 taps, unequal coarse delays in the two pols), 2 antennas, 24 spectra
    # call 2: another shape and seed, so that rows left in the shared array by call 1 would show up if they were read
    w1 = si.make_workload(1, n_spectra=24, n_antennas=2)
    w2 = si.custom_workload(A=3, n=256, T=8, S=40, seed=7, coarse_range=(-300, 700), keep_samples=False)
    got1 = _no_alloc(torch, fb, w1)
    got2 = _no_alloc(torch, fb, w2)                       # straight after call 1, same built-in array
    for w, got in ((w1, got1), (w2, got2)):
        assert np.any(got != 99)
        want, path = _existing_path(torch, fb, w)         # the kernels fengine_process picks for this shape
        _assert_same(got, want, f"{w.name} vs default path ({path})")
        want_g, path_g = _existing_path(torch, fb, w, force_generic=1)
        assert path_g == "generic"
        np.testing.assert_array_equal(got, want_g)        # the same kernels on another scratch: identical bytes
    # and once more in the other order: the array now holds call 2's rows.  By now every kernel of the entry point is
    # loaded, so the driver's free-memory figure must not move either: the call allocated nothing anywhere.
    free_before = torch.cuda.mem_get_info()[0]
    again = _no_alloc(torch, fb, w1, keep=True)
    assert torch.cuda.mem_get_info()[0] == free_before
    np.testing.assert_array_equal(again, got1)


def test_no_alloc_entry_point_refuses_what_does_not_fit(torch, fb):
    # one more spectrum than the built-in array holds for this shape: refused with a message that names the limit,
    # before any kernel runs (the output keeps its fill value)
    n, T, A, P = 64, 4, 1, 2
    N = 2 * n
    fits = fb.NOALLOC_MAX_FLOATS // (A * P * N)
    S = fits + 1
    z = lambda count, dtype: torch.zeros(count, dtype=dtype, device="cuda")
    d_in = z(A * P * N * (S + T - 1) * 10 // 8, torch.uint8)
    d_out = torch.full((A, S, n, P, 2), 99, dtype=torch.int8, device="cuda")
    tables = (z(N * T, torch.float32), z(A * P, torch.int32), z(A * P, torch.float32), z(A * P, torch.float32),
              z(A * P * n * 2, torch.float32))
    with pytest.raises(fb.FEngineError) as e:
        fb.process_noalloc(d_in, d_out, *tables, A, n, T, P, S)
    assert e.value.code == 1 and "FENGINE_NOALLOC_MAX_FLOATS" in str(e.value) and "split the batch" in str(e.value)
    torch.cuda.synchronize()
    assert bool((d_out == 99).all())
    # the largest batch that fits is accepted (zero weights and gains: every output is 0)
    fb.process_noalloc(d_in, d_out, *tables, A, n, T, P, fits)
    torch.cuda.synchronize()
    assert bool((d_out[:, :fits] == 0).all()) and bool((d_out[:, fits:] == 99).all())
