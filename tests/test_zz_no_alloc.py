"""nbk_calc_noalloc_dev -- the force call for callers that are not allowed to allocate device memory.

Some users of this library cannot call cudaMalloc: a plug-in living inside a process whose memory pool
already owns the GPU's memory, a step loop that must not be stalled by the driver's allocation lock, a code
with a "nothing is allocated after start-up" rule.  nbk_open is closed to them (it allocates); this one
context-free call keeps its split-j partial rows in a fixed 4 MiB array inside the library's device image
instead (include/nbk.h has the limits: n_i <= 4096, n_j <= 16 M, no overlapping calls).

The GPU test checks it against the path every other test uses (context: set_j -> set_ti -> firsthalf ->
lasthalf) on the same seeded particles, with the tolerances of tests/parity.py, on two calls in a row: the
second call has a different shape, so it finds the first call's rows and counters in the shared array and
must not be disturbed by them.  It runs in the default torch stream, one call after the other -- the only use
the entry point allows.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests of the main path.  The test holds no state of its own, so it passes alone in a fresh process
(where its first call also does the per-device address look-up) and after all the other tests.
"""
import ctypes

import numpy as np
import pytest

from paper_0707_0438_b200 import binding as nb
from paper_0707_0438_b200 import inputs
from parity import assert_parity

EPS = inputs.EPS_PAPER
FULL = nb.NBK_JERK | nb.NBK_POT


def _context_path(m, x, v, idx, eps2, flags):
    """The existing path: a context that owns (and allocates) its buffers."""
    n = m.shape[0]
    ctx = nb.nbk_open(0, n, max(len(idx), 1))
    try:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf(ctx, n, len(idx), idx, None, None, eps2, flags)
        return nb.nbk_calc_lasthalf(ctx, len(idx))
    finally:
        nb.nbk_close(ctx)


def _noalloc_path(torch, m, x, v, idx, eps2, flags):
    """The new entry point: every buffer is the caller's (torch tensors here), nothing is allocated inside."""
    dev = torch.device("cuda:0")
    dm, dx, dv = (torch.from_numpy(a).to(dev) for a in (m, x, v))
    di = torch.from_numpy(idx).to(dev)
    n_i = len(idx)
    # poison the outputs: every element must be written by the call
    acc = torch.full((n_i, 3), float("nan"), device=dev)
    jerk = torch.full((n_i, 3), float("nan"), device=dev)
    pot = torch.full((n_i,), float("nan"), device=dev)
    stream = torch.cuda.current_stream(dev).cuda_stream
    nb.nbk_calc_noalloc_dev(0, stream, m.shape[0], dm.data_ptr(), dx.data_ptr(), dv.data_ptr(), n_i,
                            di.data_ptr(), eps2, flags, acc.data_ptr(), jerk.data_ptr(), pot.data_ptr())
    torch.cuda.synchronize(dev)
    return acc.cpu().numpy(), jerk.cpu().numpy(), pot.cpu().numpy()


@pytest.mark.gpu
def test_noalloc_matches_context_path_on_two_calls_in_a_row():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests have no fallback")
    nb.load()
    # call 1: a block of 1000 active particles of N = 5000 (ragged i-tile, ragged j-tile, several j-splits)
    # call 2: all of N = 1531 at eps = 0 (other i-tile and split counts; the zero-distance mask; stale rows
    #         and counters of call 1 are in the array)
    cases = [(5000, 1000, np.float32(EPS) ** 2, FULL, 11),
             (1531, 1531, np.float32(0.0), FULL | nb.NBK_EPS0, 12)]
    first = None
    for n, n_i, eps2, flags, seed in cases:
        m, x, v = inputs.plummer_f32(n, seed=seed)
        idx = np.ascontiguousarray(inputs.active_block(n, n_i, seed=seed), dtype=np.int32)
        want = _context_path(m, x, v, idx, eps2, flags)
        got = _noalloc_path(torch, m, x, v, idx, eps2, flags)
        assert_parity(got, want, what=f"noalloc n={n} n_i={n_i} eps2={eps2}")
        if first is None:
            first = (m, x, v, idx, eps2, flags, got)
    # call 3: the first problem again, after another shape used the array -- same bits as before
    m, x, v, idx, eps2, flags, got1 = first
    again = _noalloc_path(torch, m, x, v, idx, eps2, flags)
    for a, b in zip(got1, again):
        assert np.array_equal(a, b), "the shared scratch array leaked state from one call into the next"


@pytest.mark.gpu
def test_noalloc_without_jerk_and_with_identity_index():
    """acc + pot only (v and i_index NULL): jerk reads zero, as after a lasthalf without NBK_JERK."""
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests have no fallback")
    nb.load()
    m, x, v = inputs.plummer_f32(777, seed=5)
    idx = np.arange(777, dtype=np.int32)
    eps2 = np.float32(EPS) ** 2
    want = _context_path(m, x, v, idx, eps2, nb.NBK_POT)
    dev = torch.device("cuda:0")
    dm, dx = torch.from_numpy(m).to(dev), torch.from_numpy(x).to(dev)
    acc = torch.full((777, 3), float("nan"), device=dev)
    jerk = torch.full((777, 3), float("nan"), device=dev)
    pot = torch.full((777,), float("nan"), device=dev)
    nb.nbk_calc_noalloc_dev(0, torch.cuda.current_stream(dev).cuda_stream, 777, dm.data_ptr(), dx.data_ptr(), 0,
                            777, 0, eps2, nb.NBK_POT, acc.data_ptr(), jerk.data_ptr(), pot.data_ptr())
    torch.cuda.synchronize(dev)
    assert_parity((acc.cpu().numpy(), jerk.cpu().numpy(), pot.cpu().numpy()), want, jerk=False, what="noalloc acc+pot")
    assert torch.all(jerk == 0)


def test_noalloc_refuses_sizes_beyond_its_fixed_array():
    """Argument checks come before any CUDA call, so they hold on a box without a GPU too: a size the fixed
    array cannot serve is NBK_ERANGE with a message that says so, never a silent overrun."""
    lib = nb.load()
    err = ctypes.c_int(123)
    one = ctypes.c_void_p(256)  # never dereferenced: the call is refused first
    args_tail = (one, 0.0, FULL, one, one, one, ctypes.byref(err))
    assert lib.nbk_calc_noalloc_dev(0, None, 1000, one, one, one, nb.NBK_NOALLOC_MAX_NI + 1, *args_tail) == nb.NBK_ERANGE
    assert lib.nbk_calc_noalloc_dev(0, None, nb.NBK_NOALLOC_MAX_NJ + 1, one, one, one, 16, *args_tail) == nb.NBK_ERANGE
    assert err.value == 0
    assert lib.nbk_calc_noalloc_dev(0, None, -1, one, one, one, 16, *args_tail) == nb.NBK_EINVAL
    assert lib.nbk_calc_noalloc_dev(-1, None, 16, one, one, one, 16, *args_tail) == nb.NBK_EINVAL
    assert lib.nbk_calc_noalloc_dev(0, None, 16, one, one, None, 16, *args_tail) == nb.NBK_EINVAL  # NBK_JERK needs v
    assert lib.nbk_calc_noalloc_dev(0, None, 16, one, one, one, 16, one, 0.0, FULL | nb.NBK_NN, one, one, one,
                                    None) == nb.NBK_EINVAL
    assert lib.nbk_calc_noalloc_dev(0, None, 16, one, one, one, 16, one, -1.0, FULL, one, one, one, None) == nb.NBK_EINVAL
    assert lib.nbk_calc_noalloc_dev(0, None, 16, one, one, one, 0, *args_tail) == nb.NBK_OK  # nothing to do
    with pytest.raises(nb.NbkError, match="out of range"):
        nb.nbk_calc_noalloc_dev(0, 0, 16, 256, 256, 256, nb.NBK_NOALLOC_MAX_NI + 1, 256, 0.0, FULL, 256, 256, 256)
