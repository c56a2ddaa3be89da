"""GPU parity of the j-sharded path (include/nbk.h "j-sharding") against the
fp64 oracle on the whole system.  The box has one GPU, so the G shards are G contexts of one
process run one after the other (no kernel waits on another); the two all-reduces are replaced, in
the test only, by a sum over the G buffers.  What is under test is the kernel side: ownership
mapping, zero-filled state exchange, external i-state with the own entry left out by local address,
fp64 partial sums, the single rounding."""
import numpy as np
import pytest

from paper_0707_0438_b200 import binding as nb
from paper_0707_0438_b200 import inputs
from paper_0707_0438_b200.sharded import ShardedForce, shard_bounds
from parity import assert_parity

pytestmark = pytest.mark.gpu

EPS = inputs.EPS_PAPER
FULL = nb.NBK_JERK | nb.NBK_POT


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests have no fallback")
    nb.load()
    return torch


def run_shards(torch, world, m, x, v, eps, ii, flags=FULL, tj=None, a=None, k=None, t=0.0, peer=False):
    """G contexts on one GPU, run in turn; sums over the G buffers stand in for the all-reduces."""
    n, n_i = m.shape[0], ii.shape[0]
    dev = torch.device("cuda", 0)
    ts = torch.cuda.Stream(device=dev)   # one stream for the G contexts and the torch sums between them
    stream = ts.cuda_stream
    ig = torch.from_numpy(ii.astype(np.int32)).to(dev)
    torch.cuda.synchronize()
    with torch.cuda.stream(ts):
        return _run_shards_on(torch, dev, stream, ig, world, m, x, v, eps, ii, flags, tj, a, k, t, peer)


def _run_shards_on(torch, dev, stream, ig, world, m, x, v, eps, ii, flags, tj, a, k, t, peer):
    n, n_i = m.shape[0], ii.shape[0]
    ctxs, bounds = [], []
    for r in range(world):
        j0, j1 = shard_bounds(n, world, r)
        c = nb.nbk_open(0, max(j1 - j0, 1), max(n_i, 1), stream)
        if j1 > j0:
            cut = lambda arr: None if arr is None else arr[j0:j1]
            nb.nbk_set_j_particles(c, None, cut(tj), m[j0:j1], x[j0:j1], v[j0:j1], cut(a), cut(k))
        nb.nbk_set_ti(c, t)
        ctxs.append(c)
        bounds.append((j0, j1))
    try:
        il = [torch.empty(n_i, dtype=torch.int32, device=dev) for _ in range(world)]
        xv = [torch.empty((n_i, 8), dtype=torch.float32, device=dev) for _ in range(world)]
        for r, c in enumerate(ctxs):
            j0, j1 = bounds[r]
            nb.nbk_shard_gather_i_dev(c, j1 - j0, j0, n_i, ig.data_ptr(), il[r].data_ptr(), xv[r].data_ptr())
        owners = torch.stack([(t_ >= 0).to(torch.int32) for t_ in il]).sum(0)
        assert bool((owners == 1).all()), "every i-particle has exactly one owner"
        s64 = [torch.empty((n_i, 8), dtype=torch.float64, device=dev) for _ in range(world)]
        acc = torch.empty((n_i, 3), dtype=torch.float32, device=dev)
        jerk = torch.empty((n_i, 3), dtype=torch.float32, device=dev)
        pot = torch.empty(n_i, dtype=torch.float32, device=dev)
        if peer:   # the peer-memory form: every "rank" reads the others' buffers by pointer; the stream
            begin = [b[0] for b in bounds] + [n]   # order of this one process stands in for the barriers
            xvf = [torch.empty((n_i, 8), dtype=torch.float32, device=dev) for _ in range(world)]
            for r, c in enumerate(ctxs):
                nb.nbk_shard_fetch_i_dev(c, n_i, ig.data_ptr(), begin, [t_.data_ptr() for t_ in xv], xvf[r].data_ptr())
            for r, c in enumerate(ctxs):
                j0, j1 = bounds[r]
                nb.nbk_shard_calc_partial_dev(c, j1 - j0, n_i, il[r].data_ptr(), xvf[r].data_ptr(),
                                              np.float32(eps) ** 2, flags, s64[r].data_ptr())
            outs = []
            for r, c in enumerate(ctxs):   # every rank combines for itself: all must get the same bits
                o = [torch.empty_like(acc), torch.empty_like(jerk), torch.empty_like(pot)]
                nb.nbk_shard_combine_dev(c, n_i, [t_.data_ptr() for t_ in s64], *[t_.data_ptr() for t_ in o])
                outs.append(o)
            torch.cuda.synchronize()
            for o in outs[1:]:
                assert all(torch.equal(p_, q_) for p_, q_ in zip(o, outs[0]))
            acc, jerk, pot = outs[0]
            xv_all = xvf[world - 1]
            return acc.cpu().numpy(), jerk.cpu().numpy(), pot.cpu().numpy(), xv_all.cpu().numpy()
        xv_all = torch.stack(xv).sum(0).contiguous()       # stands in for all-reduce #1
        for r, c in enumerate(ctxs):
            j0, j1 = bounds[r]
            nb.nbk_shard_calc_partial_dev(c, j1 - j0, n_i, il[r].data_ptr(), xv_all.data_ptr(),
                                          np.float32(eps) ** 2, flags, s64[r].data_ptr())
        tot = torch.stack(s64).sum(0).contiguous()         # stands in for all-reduce #2
        nb.nbk_shard_finish_dev(ctxs[0], n_i, tot.data_ptr(), acc.data_ptr(), jerk.data_ptr(), pot.data_ptr())
        torch.cuda.synchronize()
        return acc.cpu().numpy(), jerk.cpu().numpy(), pot.cpu().numpy(), xv_all.cpu().numpy()
    finally:
        for c in ctxs:
            nb.nbk_close(c)


@pytest.mark.parametrize("world", [1, 2, 3, 8])
@pytest.mark.parametrize("n,n_i", [(16384, 16384), (16384, 37), (4099, 1031)])
def test_sharded_parity_vs_whole_system_oracle(gpu, c_oracle, world, n, n_i):
    m, x, v = inputs.plummer_f32(n, 2)
    ii = np.arange(n, dtype=np.int32) if n_i == n else inputs.active_block(n, n_i, 21)
    ref = c_oracle.force(m, x, v, EPS, i_index=ii)
    acc, jerk, pot, xv = run_shards(gpu, world, m, x, v, EPS, ii)
    assert np.array_equal(xv[:, 0:3], x[ii]) and np.array_equal(xv[:, 4:7], v[ii])   # exact copy
    assert_parity((acc, jerk, pot), ref, what=f"sharded G={world} n={n} n_i={n_i}")


@pytest.mark.parametrize("world", [1, 3, 8, 16])
def test_sharded_peer_memory_form_parity_and_same_bits_as_collective_form(gpu, c_oracle, world):
    """nbk_shard_fetch_i_dev / nbk_shard_combine_dev (P2P loads by pointer) against the oracle, and
    bit for bit against the collective form: both add the ranks' fp64 rows in rank order."""
    n, n_i = 4099, 1031
    m, x, v = inputs.plummer_f32(n, 2)
    ii = inputs.active_block(n, n_i, 21)
    ref = c_oracle.force(m, x, v, EPS, i_index=ii)
    got = run_shards(gpu, world, m, x, v, EPS, ii, peer=True)
    assert np.array_equal(got[3][:, 0:3], x[ii]) and np.array_equal(got[3][:, 4:7], v[ii])
    assert_parity(got[:3], ref, what=f"peer-memory G={world}")
    coll = run_shards(gpu, world, m, x, v, EPS, ii, peer=False)
    for g, c in zip(got[:3], coll[:3]):
        assert np.array_equal(g, c)


def test_sharded_eps0_and_acc_only(gpu, c_oracle):
    n = 8192
    m, x, v = inputs.plummer_f32(n, 7)
    ii = inputs.active_block(n, 2048, 22)
    ref = c_oracle.force(m, x, v, 0.0, i_index=ii)
    acc, jerk, pot, _ = run_shards(gpu, 4, m, x, v, 0.0, ii, flags=FULL | nb.NBK_EPS0)
    assert_parity((acc, jerk, pot), ref, what="sharded eps=0")
    ref = c_oracle.force(m, x, v, EPS, i_index=ii, want_jerk=False)
    acc, jerk, pot, _ = run_shards(gpu, 4, m, x, v, EPS, ii, flags=nb.NBK_POT)
    assert_parity((acc, jerk, pot), ref, jerk=False, what="sharded acc+pot")
    assert not jerk.any()


def test_sharded_with_prediction_and_more_ranks_than_particles(gpu, c_oracle):
    """Predicted state is what is exchanged; shards may be empty (G > n)."""
    n, t = 5, 0.01
    m, x, v = inputs.plummer_f32(n, 9)
    a, k = inputs.gaussian_derivatives(n, 10)
    tj = inputs.particle_times(n, t, 11)
    ii = np.arange(n, dtype=np.int32)
    xp, vp = c_oracle.predict(t, tj, x, v, a, k)
    xp, vp = xp.astype(np.float32), vp.astype(np.float32)
    ref = c_oracle.force(m, xp, vp, EPS, i_index=ii)
    acc, jerk, pot, xv = run_shards(gpu, 8, m, x, v, EPS, ii, tj=tj, a=a, k=k, t=t)
    assert np.max(np.abs(xv[:, 0:3] - xp)) <= 1.2e-7 * np.max(np.abs(xp))
    assert_parity((acc, jerk, pot), ref, what="sharded G=8 n=5")


def test_sharded_world1_class_equals_plain_path_bitwise(gpu, c_oracle):
    """ShardedForce at world size 1 (no collective): same bits as firsthalf/lasthalf, because the
    fp64 sums are rounded once either way."""
    n, n_i = 16384, 2048
    m, x, v = inputs.plummer_f32(n, 2)
    ii = inputs.active_block(n, n_i, 23)
    sf = ShardedForce(n, n_i, device=0)
    try:
        assert (sf.world, sf.j0, sf.j1) == (1, 0, n)
        sf.set_j_particles(None, None, m, x, v)
        sf.set_ti(0.0)
        ig = gpu.from_numpy(ii).to("cuda:0")
        acc, jerk, pot = sf.calc(ig, np.float32(EPS) ** 2)
        gpu.cuda.synchronize()
        got = (acc.cpu().numpy(), jerk.cpu().numpy(), pot.cpu().numpy())
        assert sf.collectives == 0
    finally:
        sf.close()
    c = nb.nbk_open(0, n, n_i)
    try:
        nb.nbk_set_j_particles(c, None, None, m, x, v)
        nb.nbk_set_ti(c, 0.0)
        nb.nbk_calc_firsthalf(c, n, n_i, ii, None, None, np.float32(EPS) ** 2, FULL)
        plain = nb.nbk_calc_lasthalf(c, n_i)
    finally:
        nb.nbk_close(c)
    for g, p in zip(got, plain):
        assert np.array_equal(g, p)
    assert_parity(got, c_oracle.force(m, x, v, EPS, i_index=ii), what="ShardedForce world 1")


NCCL_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import numpy as np, torch
import torch.distributed as dist
from paper_0707_0438_b200 import binding as nb, inputs
from paper_0707_0438_b200.sharded import ShardedForce
torch.cuda.set_device(0)
dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
n, n_i = 16384, 4096
m, x, v = inputs.plummer_f32(n, 2)
ii = inputs.active_block(n, n_i, 24)
e2 = float(np.float32(inputs.EPS_PAPER) ** 2)
sf = ShardedForce(n, n_i, device=0, always_reduce=True)
sf.set_j_particles(None, None, m, x, v)
sf.set_ti(0.0)
ig = torch.from_numpy(ii).to("cuda:0")
outs = [tuple(t.clone() for t in sf.calc(ig, e2)) for _ in range(3)]
torch.cuda.synchronize()
assert sf.collectives == 6
c = nb.nbk_open(0, n, n_i)
nb.nbk_set_j_particles(c, None, None, m, x, v)
nb.nbk_set_ti(c, 0.0)
nb.nbk_calc_firsthalf(c, n, n_i, ii, None, None, e2, nb.NBK_JERK | nb.NBK_POT)
plain = nb.nbk_calc_lasthalf(c, n_i)
nb.nbk_close(c)
for o in outs:
    for g, p in zip(o, plain):
        assert np.array_equal(g.cpu().numpy(), p)
sf.close()
si = ShardedForce(n, n_i, device=0, always_reduce=True, mode="i")   # i-sharding: three all-gathers per call
si.set_j_particles(None, None, m, x, v)
si.set_ti(0.0)
for rep in range(2):
    o = si.calc(ig, e2)
    torch.cuda.synchronize()
    for g, p in zip(o, plain):
        assert np.array_equal(g.cpu().numpy(), p)
assert si.collectives == 6
si.close()
dist.destroy_process_group()
print("NCCL_OK")
"""


def test_sharded_class_with_nccl_collectives_at_world1(gpu, tmp_path):
    """The real collectives (NCCL all-reduce of fp32 state and fp64 sums on the library's stream) at
    world size 1, where a sum over ranks is the identity: results equal the plain path bit for bit."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "nccl_worker.py"
    script.write_text(NCCL_WORKER.format(root=root))
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
    p = subprocess.run([sys.executable, str(script)], env=env, capture_output=True, text=True, timeout=600)
    assert p.returncode == 0 and "NCCL_OK" in p.stdout, p.stdout + p.stderr


def test_i_sharded_world1_class_equals_plain_path_bitwise(gpu, c_oracle):
    """mode="i" at world size 1: the slice is the whole i-list, so the results are the plain path's."""
    n, n_i = 8192, 1000
    m, x, v = inputs.plummer_f32(n, 4)
    ii = inputs.active_block(n, n_i, 25)
    sf = ShardedForce(n, n_i, device=0, mode="i")
    try:
        sf.set_j_particles(None, None, m, x, v)
        sf.set_ti(0.0)
        ig = gpu.from_numpy(ii).to("cuda:0")
        out = (gpu.empty((n_i, 3), device="cuda:0"), gpu.empty((n_i, 3), device="cuda:0"), gpu.empty(n_i, device="cuda:0"))
        got = sf.calc(ig, np.float32(EPS) ** 2, out=out)
        gpu.cuda.synchronize()
        got = tuple(t.cpu().numpy() for t in got)
        view = sf.calc(ig, np.float32(EPS) ** 2)
        gpu.cuda.synchronize()
        for g, w in zip(got, view):
            assert np.array_equal(g, w.cpu().numpy())
        assert sf.collectives == 0
    finally:
        sf.close()
    assert_parity(got, c_oracle.force(m, x, v, EPS, i_index=ii), what="i-sharded world 1")


PEER_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import numpy as np, torch
import torch.distributed as dist
from paper_0707_0438_b200 import binding as nb, inputs
from paper_0707_0438_b200.sharded import ShardedForce
torch.cuda.set_device(0)
dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
n, n_i = 16384, 4096
m, x, v = inputs.plummer_f32(n, 2)
ii = inputs.active_block(n, n_i, 24)
e2 = float(np.float32(inputs.EPS_PAPER) ** 2)
try:   # platform capability: symmetric memory allocation and rendezvous
    import torch.distributed._symmetric_memory as symm_mem
    probe = symm_mem.empty((1024,), dtype=torch.uint8, device=torch.device("cuda", 0))
    symm_mem.rendezvous(probe, dist.group.WORLD)
except Exception as e:
    print("SYMM_UNAVAILABLE", type(e).__name__, str(e)[:200])
    dist.destroy_process_group()
    sys.exit(0)
sp = ShardedForce(n, n_i, device=0, transport="peer")   # symmetric memory + barriers + P2P kernels
sp.set_j_particles(None, None, m, x, v)
sp.set_ti(0.0)
ig = torch.from_numpy(ii).to("cuda:0")
outs = [tuple(t.clone() for t in sp.calc(ig, e2)) for _ in range(3)]
torch.cuda.synchronize()
assert sp.barriers == 6 and sp.collectives == 0
c = nb.nbk_open(0, n, n_i)
nb.nbk_set_j_particles(c, None, None, m, x, v)
nb.nbk_set_ti(c, 0.0)
nb.nbk_calc_firsthalf(c, n, n_i, ii, None, None, e2, nb.NBK_JERK | nb.NBK_POT)
plain = nb.nbk_calc_lasthalf(c, n_i)
nb.nbk_close(c)
for o in outs:
    for g, p in zip(o, plain):
        assert np.array_equal(g.cpu().numpy(), p)
sp.close()
dist.destroy_process_group()
print("PEER_OK")
"""


def test_sharded_peer_transport_with_symmetric_memory_at_world1(gpu, tmp_path):
    """transport="peer" with real torch symmetric memory, its barriers and the P2P kernels at world size 1:
    bit-equal to the plain path.  Skipped only if the platform cannot allocate / rendezvous symmetric memory."""
    import os
    import socket
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "peer_worker.py"
    script.write_text(PEER_WORKER.format(root=root))
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
    p = subprocess.run([sys.executable, str(script)], env=env, capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stdout + p.stderr
    if "SYMM_UNAVAILABLE" in p.stdout:
        pytest.skip("symmetric memory unavailable here: " + p.stdout.strip().splitlines()[-1])
    assert "PEER_OK" in p.stdout, p.stdout + p.stderr


def test_sharded_refused_calls(gpu):
    c = nb.nbk_open(0, 64, 64)
    try:
        buf = gpu.zeros(64 * 8, dtype=gpu.float64, device="cuda:0")
        with pytest.raises(nb.NbkError) as e:
            nb.nbk_shard_calc_partial_dev(c, 64, 8, buf.data_ptr(), buf.data_ptr(), 0.0, FULL | nb.NBK_NN,
                                          buf.data_ptr())
        assert e.value.status == nb.NBK_EINVAL
        with pytest.raises(nb.NbkError) as e:
            nb.nbk_shard_gather_i_dev(c, 65, 0, 8, buf.data_ptr(), buf.data_ptr(), buf.data_ptr())
        assert e.value.status == nb.NBK_ERANGE
        with pytest.raises(nb.NbkError) as e:
            nb.nbk_shard_calc_partial_dev(c, 64, 8, 0, buf.data_ptr(), 0.0, FULL, buf.data_ptr())
        assert e.value.status == nb.NBK_EINVAL
    finally:
        nb.nbk_close(c)
