"""Out-of-bounds writes, looked for with guard bands (compute-sanitizer is closed on this GPU pool:
profiles/r03_sanitizer.md).

nbk_open_ws puts EVERY device buffer of a context (j-state, predicted arrays, i-staging, partial rows, results,
counters, neighbour buffers) into one caller-owned workspace, and the _dev calls write their results into
caller-owned arrays.  Here the workspace and the result arrays each sit between two 1 MiB bands of a byte
pattern; every launch shape of the force path runs (all i-per-thread forms, one-launch and two-launch small
blocks, neighbour search and its re-scan kernel, eps = 0, external i-particles, scatter by address, the
predictor at a later time) and the bands must come out untouched, and so must the part of each result array
beyond n_i.  A kernel that indexes past the end (or before the start) of the memory it was given lands in a
band.  It cannot see a write that stays inside the workspace but in the wrong sub-buffer: the element-wise
parity tests are what catch those.
"""
import numpy as np
import pytest

from paper_0707_0438_b200 import binding as nb
from paper_0707_0438_b200 import inputs
from parity import assert_parity

pytestmark = pytest.mark.gpu

EPS = inputs.EPS_PAPER
FULL = nb.NBK_JERK | nb.NBK_POT
BAND = 1 << 20
PATTERN = 0xA5


class Banded:
    """`nbytes` of device memory between two pattern-filled bands (torch owns the memory)."""

    def __init__(self, torch, nbytes):
        self.torch = torch
        self.nbytes = int(nbytes)
        pad = (-self.nbytes) % 256
        self.arena = torch.full((BAND + self.nbytes + pad + BAND,), PATTERN, dtype=torch.uint8, device="cuda")
        assert self.arena.data_ptr() % 256 == 0
        self.ptr = self.arena.data_ptr() + BAND

    def inner(self):
        return self.arena[BAND:BAND + self.nbytes]

    def bands_intact(self):
        lo = self.arena[:BAND]
        hi = self.arena[BAND + self.nbytes:]
        return bool((lo == PATTERN).all().item()) and bool((hi == PATTERN).all().item())


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests have no fallback")
    nb.load()
    return torch


def test_no_kernel_writes_outside_the_workspace_or_the_result_arrays(gpu, c_oracle):
    torch = gpu
    n = 4099                                    # ragged against every tile size
    m, x, v = inputs.plummer_f32(n, seed=404)
    ws = Banded(torch, nb.nbk_workspace_bytes(0, n, n))
    out_acc, out_jrk = Banded(torch, 4 * 3 * n), Banded(torch, 4 * 3 * n)
    out_pot, out_nn, out_r2 = Banded(torch, 4 * n), Banded(torch, 4 * n), Banded(torch, 4 * n)
    dm, dx, dv = (torch.from_numpy(t).cuda() for t in (m, x, v))
    perm = np.random.default_rng(4).permutation(n).astype(np.int32)
    dperm = torch.from_numpy(perm).cuda()
    dmp, dxp, dvp = (torch.from_numpy(np.ascontiguousarray(t[perm])).cuda() for t in (m, x, v))
    ext = inputs.plummer_f32(300, seed=405)[1]
    ref_full = c_oracle.force(m, x, v, EPS)
    ctx = nb.nbk_open_ws(0, n, n, 0, ws.ptr, ws.nbytes)
    checked = 0
    try:
        # a1 scatter by (shuffled) address from device arrays, a3 predictor
        nb.nbk_set_j_particles_dev(ctx, n, dperm.data_ptr(), 0, dmp.data_ptr(), dxp.data_ptr(), dvp.data_ptr())
        nb.nbk_set_ti(ctx, 0.0)
        shapes = [(0x00, n, FULL, EPS), (0x10, n, FULL, EPS), (0x20, n, FULL, EPS), (0x40, n, FULL, EPS),
                  (0x00, n, nb.NBK_POT, EPS), (0x00, n, FULL | nb.NBK_NN, EPS), (0x00, n, FULL, 0.0),
                  (0x00, 1, FULL, EPS), (0x00, 5, FULL, EPS), (0x00, 32, FULL, EPS), (0x100, 32, FULL, EPS),
                  (0x00, 32, FULL | nb.NBK_NN, 0.0), (0x00, 33, FULL, EPS), (0x00, 777, FULL | nb.NBK_NN, EPS),
                  (0x00, 2049, FULL, EPS)]
        for variant, n_i, flags, eps in shapes:
            nb.nbk_set_variant(ctx, variant)
            idx = None if n_i == n else inputs.active_block(n, n_i, seed=n_i)
            for o in (out_acc, out_jrk, out_pot, out_nn, out_r2):
                o.inner().fill_(PATTERN)
            nb.nbk_calc_firsthalf(ctx, n, n_i, idx, None, None, np.float32(eps) ** 2, flags)
            nb.nbk_calc_lasthalf_dev(ctx, n_i, out_acc.ptr, out_jrk.ptr, out_pot.ptr)
            if flags & nb.NBK_NN:
                nb.nbk_get_neighbours_dev(ctx, n_i, out_nn.ptr, out_r2.ptr)
            nb.nbk_sync(ctx)
            what = f"variant {variant:#x} n_i={n_i} flags={flags} eps={eps}"
            for o, per in ((out_acc, 12), (out_jrk, 12), (out_pot, 4), (out_nn, 4), (out_r2, 4)):
                assert o.bands_intact(), what
                assert bool((o.inner()[per * n_i:] == PATTERN).all().item()), what + ": wrote beyond n_i"
            assert ws.bands_intact(), what
            if n_i == n and eps == EPS and flags & nb.NBK_JERK:   # and the results are the right ones
                got = tuple(o.inner()[:k * 4 * n].view(torch.float32).cpu().numpy().reshape(shape)
                            for o, k, shape in ((out_acc, 3, (n, 3)), (out_jrk, 3, (n, 3)), (out_pot, 1, (n,))))
                assert_parity(got, ref_full, what=what)
                checked += 1
        nb.nbk_set_variant(ctx, 0)
        # external i-particles with explicit positions, and the predictor at a later time
        nb.nbk_set_ti(ctx, 0.015625)
        nb.nbk_calc_firsthalf(ctx, n, 300, np.full(300, -1, np.int32), ext, None, np.float32(EPS) ** 2, FULL)
        nb.nbk_calc_lasthalf_dev(ctx, 300, out_acc.ptr, out_jrk.ptr, out_pot.ptr)
        nb.nbk_sync(ctx)
        assert ws.bands_intact() and out_acc.bands_intact() and out_jrk.bands_intact() and out_pot.bands_intact()
    finally:
        nb.nbk_close(ctx)
    assert checked >= 5
    assert ws.bands_intact()
