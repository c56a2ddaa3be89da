"""Host logic of the j-sharded path (paper_0707_0438_b200/sharded.py) at
world size 2 on the CPU over gloo.  The three device steps are replaced, in this test only, by an
`ops` object built on the oracle restricted to the rank's j-shard; what is under test is the
shard bounds, the local address mapping, the zero-filled state exchange, the two all-reduces and
that every rank ends with the same bits -- against the oracle on the whole system."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_0707_0438_b200.sharded import shard_bounds  # noqa: E402

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import numpy as np, torch
import torch.distributed as dist
from oracle import nbody_oracle as O
from paper_0707_0438_b200 import inputs
from paper_0707_0438_b200.sharded import ShardedForce

class OracleOps:   # test stand-in for the three device steps: oracle on the local j-shard
    def __init__(self, cap):
        z = lambda *s: np.zeros(s)
        self.m, self.t = z(cap), z(cap)
        self.x, self.v, self.a, self.k = z(cap, 3), z(cap, 3), z(cap, 3), z(cap, 3)
        self.ti = 0.0
    def alloc(self, shape, dtype):
        return torch.zeros(shape, dtype=dtype)
    def set_j_local(self, addr, tj, m, x, v, a, jerk):
        self.m[addr] = m; self.x[addr] = x
        self.t[addr] = 0.0 if tj is None else tj
        for dst, src in ((self.v, v), (self.a, a), (self.k, jerk)):
            dst[addr] = 0.0 if src is None else src
    def set_ti(self, t):
        self.ti = t
    def _pred(self, n):
        xp, vp = O.predict(self.ti, self.t[:n], self.x[:n], self.v[:n], self.a[:n], self.k[:n])
        return xp.astype(np.float32), vp.astype(np.float32)
    def gather_i(self, n_local, j0, n_i, i_global, i_local, xv):
        xp, vp = self._pred(n_local)
        g = i_global.numpy().astype(np.int64) - j0
        mine = (g >= 0) & (g < n_local)
        i_local.copy_(torch.from_numpy(np.where(mine, g, -1).astype(np.int32)))
        out = np.zeros((n_i, 8), np.float32)
        out[mine, 0:3] = xp[g[mine]]; out[mine, 4:7] = vp[g[mine]]
        xv.copy_(torch.from_numpy(out))
    def calc_partial(self, n_local, n_i, i_local, xv, eps2, flags, sum64):
        xp, vp = self._pred(n_local)
        s = np.zeros((n_i, 8))
        if n_local:
            xvn = xv.numpy()
            acc, jrk, pot = O.force(self.m[:n_local].astype(np.float32), xp, vp, np.sqrt(eps2),
                                    i_index=i_local.numpy(), xi=xvn[:, 0:3], vi=xvn[:, 4:7])
            s[:, 0:3] = acc; s[:, 3] = -pot; s[:, 4:7] = jrk
        sum64.copy_(torch.from_numpy(s))
    def calc_slice(self, n_j, i_index, eps2, flags, acc, jerk, pot):
        xp, vp = self._pred(n_j)
        a_, j_, p_ = O.force(self.m[:n_j].astype(np.float32), xp, vp, np.sqrt(eps2), i_index=i_index.numpy())
        acc.copy_(torch.from_numpy(a_.astype(np.float32)))
        jerk.copy_(torch.from_numpy(j_.astype(np.float32)))
        pot.copy_(torch.from_numpy(p_.astype(np.float32)))
    def finish(self, n_i, sum64, acc, jerk, pot):
        s = sum64.numpy()
        acc.copy_(torch.from_numpy(s[:, 0:3].astype(np.float32)))
        jerk.copy_(torch.from_numpy(s[:, 4:7].astype(np.float32)))
        pot.copy_(torch.from_numpy((-s[:, 3]).astype(np.float32)))

rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
n, n_i, eps, t = {n}, {n_i}, 1.0 / 256.0, 0.01
m, x, v = inputs.plummer_f32(n, 11)
a, k = inputs.gaussian_derivatives(n, 12)
tj = inputs.particle_times(n, t, 13)
mode = {mode!r}
sf = ShardedForce(n, n_i, ops=OracleOps(n + 1 if mode == "i" else (n + world - 1) // world + 1), mode=mode)
kept = sf.set_j_particles(None, tj, m, x, v, a, k)
sf.set_ti(t)
ii = inputs.active_block(n, n_i, 14).astype(np.int32)
acc, jerk, pot = (t.clone() for t in sf.calc(torch.from_numpy(ii), eps * eps))
# a second call after updating two particles owned by different ranks (global addresses 1 and n-2)
upd = np.array([1, n - 2])
sf.set_j_particles(upd, np.full(2, t), m[upd], x[upd] + np.float32(0.25), v[upd], a[upd], k[upd])
acc2, jerk2, pot2 = sf.calc(torch.from_numpy(ii), eps * eps)
dist.barrier()
dist.destroy_process_group()
print(json.dumps(dict(rank=rank, j0=sf.j0, j1=sf.j1, kept=kept, collectives=sf.collectives,
                      acc=acc.numpy().tolist(), jerk=jerk.numpy().tolist(), pot=pot.numpy().tolist(),
                      acc2=acc2.numpy().tolist(), pot2=pot2.numpy().tolist())))
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_shard_bounds_cover_and_balance():
    for n in (0, 1, 7, 1024, 131072, 1000003):
        for world in (1, 2, 3, 8):
            cuts = [shard_bounds(n, world, r) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            assert all(cuts[r][1] == cuts[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in cuts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_bounds(10, 2, 2)


@pytest.mark.parametrize("mode", ["j", "i"])
def test_sharded_force_world2_matches_whole_system_oracle(tmp_path, mode):
    from oracle import nbody_oracle as O
    from paper_0707_0438_b200 import inputs
    from parity import assert_parity

    n, n_i = 301, 97   # odd sizes: unequal shards, i-particles owned by both ranks
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT, n=n, n_i=n_i, mode=mode))
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=300)
        assert p.returncode == 0, err
        outs.append(json.loads(out.strip().splitlines()[-1]))
    outs.sort(key=lambda o: o["rank"])
    if mode == "j":
        assert (outs[0]["j0"], outs[0]["j1"], outs[1]["j0"], outs[1]["j1"]) == (0, 150, 150, 301)
        assert outs[0]["kept"] == 150 and outs[1]["kept"] == 151
        assert outs[0]["collectives"] == 4 and outs[1]["collectives"] == 4   # two all-reduces per call
    else:   # j replicated, i-list cut in two (49 + 48 of 97), three all-gathers per call
        assert (outs[0]["j0"], outs[0]["j1"], outs[1]["j0"], outs[1]["j1"]) == (0, 301, 0, 301)
        assert outs[0]["kept"] == 301 and outs[1]["kept"] == 301
        assert outs[0]["collectives"] == 6 and outs[1]["collectives"] == 6
    for key in ("acc", "jerk", "pot", "acc2", "pot2"):   # an all-reduce gives every rank the same bits
        assert outs[0][key] == outs[1][key], key

    eps, t = 1.0 / 256.0, 0.01
    m, x, v = inputs.plummer_f32(n, 11)
    a, k = inputs.gaussian_derivatives(n, 12)
    tj = inputs.particle_times(n, t, 13)
    ii = inputs.active_block(n, n_i, 14)
    xp, vp = O.predict(t, tj, x, v, a, k)
    xp, vp = xp.astype(np.float32), vp.astype(np.float32)
    ref = O.force(m, xp, vp, eps, i_index=ii)
    got = (np.array(outs[0]["acc"]), np.array(outs[0]["jerk"]), np.array(outs[0]["pot"]))
    e = assert_parity(got, ref, what="sharded world 2")
    assert e["acc_max"] < 1e-6 and e["pot_max"] < 1e-6   # fp64 partials, one rounding

    upd = np.array([1, n - 2])
    x2, tj2 = x.copy(), tj.copy()
    x2[upd] += np.float32(0.25)
    tj2[upd] = t
    xp2, vp2 = O.predict(t, tj2, x2, v, a, k)
    ref2 = O.force(m, xp2.astype(np.float32), vp2.astype(np.float32), eps, i_index=ii)
    np.testing.assert_allclose(np.array(outs[0]["acc2"]), ref2[0], rtol=2e-6, atol=1e-9)
    np.testing.assert_allclose(np.array(outs[0]["pot2"]), ref2[2], rtol=1e-6)


def test_sharded_force_refuses_world2_without_process_group():
    from paper_0707_0438_b200.sharded import ShardedForce
    with pytest.raises(RuntimeError):
        ShardedForce(100, 10, world=2, rank=0, ops=object())
