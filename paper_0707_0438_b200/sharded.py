"""j-sharded force evaluation over several GPUs, one process per GPU.

PAPER.md L112-L118 cuts the j-particles into parts, computes partial forces per part and sums
them afterwards; here the parts live on different GPUs.  Rank r of G holds the j-particles with
global addresses [j0_r, j1_r) in its own nbk context; a force call on a block of i-particles is

    gather_i      (kernel)   owners publish the predicted i-state, zeros elsewhere
    all-reduce    (NCCL)     n_i x 8 fp32: an exact copy from the owner to every rank
    calc_partial  (kernels)  force kernel + split-j reduce against the local j-particles
    all-reduce    (NCCL)     n_i x 8 fp64 partial sums
    finish        (kernel)   one rounding to fp32

mode="i" is the other cut of SURVEY.md 8(e): every rank holds all j-particles, takes a slice of
each i-list through the ordinary firsthalf/lasthalf calls, and the result arrays are all-gathered
(no partial sums; suited to full evaluations at large N, e.g. config C4).

transport="peer" (mode "j") replaces the two all-reduces by loads from peer memory: the exchange
buffers live in torch symmetric memory mapped into every rank, a cross-rank barrier separates the
steps, `nbk_shard_fetch_i_dev` reads each i-particle's state from its owner's buffer and
`nbk_shard_combine_dev` adds the ranks' fp64 rows in rank order and rounds once (all-reduce and finish
in one kernel).  It needs NVLink/NVSwitch P2P between the ranks; NCCL stays the default.

This module holds no arithmetic of the method: it computes the shard bounds, owns the exchange
buffers and strings the three C-ABI calls (include/nbk.h, "j-sharding") and the two collectives
together on one stream.  `ops` is the object that runs the three device steps; the default is
the CUDA library (there is no CPU fallback -- without libnbk.so or a GPU it raises).  The gloo
world-size-2 test on the CPU passes its own `ops`, built on the oracle, to check the host logic.
"""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist

from . import binding as B


def shard_bounds(n_total: int, world: int, rank: int) -> tuple[int, int]:
    """Contiguous, balanced: rank r owns global addresses [r n / G, (r+1) n / G)."""
    if n_total < 0 or world < 1 or not 0 <= rank < world:
        raise ValueError("shard_bounds: bad arguments")
    return (rank * n_total) // world, ((rank + 1) * n_total) // world


class NbkShardOps:
    """The three device steps through the C ABI, on one torch stream of its own (a null stream handle
    would make nbk_open create a private stream torch knows nothing about); the collectives are
    issued under the same stream, so the whole call is ordered without host synchronisation."""

    def __init__(self, device: int, n_local_max: int, ni_max: int):
        if not torch.cuda.is_available():
            raise RuntimeError("NbkShardOps needs a CUDA device (the sharded path has no CPU fallback)")
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        self.stream = torch.cuda.Stream(device=self.device)
        self.ctx = B.nbk_open(device, max(n_local_max, 1), max(ni_max, 1), self.stream.cuda_stream)

    def close(self):
        if self.ctx is not None:
            B.nbk_close(self.ctx)
            self.ctx = None

    def alloc(self, shape, dtype):
        return torch.zeros(shape, dtype=dtype, device=self.device)

    def enter(self):
        """Order the ops' stream after the caller's current stream and make it current."""
        self._outer = torch.cuda.current_stream(self.device)
        self.stream.wait_stream(self._outer)
        self._guard = torch.cuda.stream(self.stream)
        self._guard.__enter__()

    def leave(self):
        self._guard.__exit__(None, None, None)
        self._outer.wait_stream(self.stream)

    def set_j_local(self, addr, tj, m, x, v, a, jerk):
        B.nbk_set_j_particles(self.ctx, addr, tj, m, x, v, a, jerk)

    def set_ti(self, t):
        B.nbk_set_ti(self.ctx, t)

    def gather_i(self, n_local, j0, n_i, i_global, i_local, xv):
        B.nbk_shard_gather_i_dev(self.ctx, n_local, j0, n_i, i_global.data_ptr(), i_local.data_ptr(),
                                 xv.data_ptr())

    def calc_partial(self, n_local, n_i, i_local, xv, eps2, flags, sum64):
        B.nbk_shard_calc_partial_dev(self.ctx, n_local, n_i, i_local.data_ptr(), xv.data_ptr(), eps2, flags,
                                     sum64.data_ptr())

    def finish(self, n_i, sum64, acc, jerk, pot):
        B.nbk_shard_finish_dev(self.ctx, n_i, sum64.data_ptr(), acc.data_ptr(), jerk.data_ptr(), pot.data_ptr())

    def fetch_i(self, n_i, i_global, shard_begin, peer_xv, xv):
        B.nbk_shard_fetch_i_dev(self.ctx, n_i, i_global.data_ptr(), shard_begin, peer_xv, xv.data_ptr())

    def combine(self, n_i, peer_sum64, acc, jerk, pot):
        B.nbk_shard_combine_dev(self.ctx, n_i, peer_sum64, acc.data_ptr(), jerk.data_ptr(), pot.data_ptr())

    def calc_slice(self, n_j, i_index, eps2, flags, acc, jerk, pot):
        """i-sharding: the plain firsthalf / lasthalf pair on this rank's slice of the i-list."""
        n_i = int(i_index.shape[0])
        B.nbk_calc_firsthalf_dev(self.ctx, n_j, n_i, i_index.data_ptr(), 0, 0, eps2, flags)
        B.nbk_calc_lasthalf_dev(self.ctx, n_i, acc.data_ptr(), jerk.data_ptr(), pot.data_ptr())

    def sync(self):
        B.nbk_sync(self.ctx)


class ShardedForce:
    """One rank's end of the j-sharded path.  Every rank makes the same calls in the same order."""

    def __init__(self, n_total: int, ni_max: int, device: int = 0, group=None, ops=None,
                 world: int | None = None, rank: int | None = None, always_reduce: bool = False,
                 mode: str = "j", transport: str = "nccl"):
        live = dist.is_available() and dist.is_initialized()
        self.group = group
        self.world = world if world is not None else (dist.get_world_size(group) if live else 1)
        self.rank = rank if rank is not None else (dist.get_rank(group) if live else 0)
        if self.world > 1 and not live:
            raise RuntimeError("ShardedForce with world > 1 needs an initialised process group")
        if mode not in ("j", "i"):
            raise ValueError("mode must be 'j' (j-particles sharded) or 'i' (i-particles sharded, j replicated)")
        self.mode = mode
        self.n_total, self.ni_max = int(n_total), int(ni_max)
        # mode "i": every rank holds all j-particles and takes a slice of each i-list
        self.j0, self.j1 = shard_bounds(self.n_total, self.world, self.rank) if mode == "j" else (0, self.n_total)
        self.n_local = self.j1 - self.j0
        self.ops = ops if ops is not None else NbkShardOps(device, self.n_local, self.ni_max)
        if transport not in ("nccl", "peer") or (transport == "peer" and mode != "j"):
            raise ValueError("transport must be 'nccl', or 'peer' with mode 'j'")
        self.transport = transport
        self.symm = None
        if mode == "j" and transport == "peer":
            # exchange buffers in symmetric memory: every rank maps every other rank's copy and reads it
            # with P2P loads (nbk_shard_fetch_i_dev / nbk_shard_combine_dev); two barriers per call
            import torch.distributed._symmetric_memory as symm_mem
            if not live:
                raise RuntimeError("transport='peer' needs an initialised process group")
            self.i_local = self.ops.alloc((self.ni_max,), torch.int32)
            self.xv_full = self.ops.alloc((self.ni_max, 8), torch.float32)
            self.s64_off = (self.ni_max * 32 + 255) // 256 * 256
            raw = symm_mem.empty((self.s64_off + self.ni_max * 64,), dtype=torch.uint8, device=self.ops.device)
            raw.zero_()
            self.symm_raw = raw
            self.symm = symm_mem.rendezvous(raw, group if group is not None else dist.group.WORLD)
            self.xv = raw[: self.ni_max * 32].view(torch.float32).view(self.ni_max, 8)
            self.sum64 = raw[self.s64_off: self.s64_off + self.ni_max * 64].view(torch.float64).view(self.ni_max, 8)
            self.peer_base = [int(p) for p in self.symm.buffer_ptrs]
            self.shard_begin = [shard_bounds(self.n_total, self.world, r)[0] for r in range(self.world)] + [self.n_total]
        elif mode == "j":
            self.i_local = self.ops.alloc((self.ni_max,), torch.int32)
            self.xv = self.ops.alloc((self.ni_max, 8), torch.float32)
            self.sum64 = self.ops.alloc((self.ni_max, 8), torch.float64)
        else:   # gather buffers: world equal chunks, the last one padded
            self.chunk_max = -(-self.ni_max // self.world)
            rows = self.chunk_max * self.world
            self.g_acc = self.ops.alloc((rows, 3), torch.float32)
            self.g_jerk = self.ops.alloc((rows, 3), torch.float32)
            self.g_pot = self.ops.alloc((rows,), torch.float32)
        self.collectives = 0   # all-reduces / all-gathers issued so far (for tests and bench)
        self.barriers = 0      # symmetric-memory barriers issued so far (transport 'peer')
        # issue the collectives at world size 1 too (needs a process group): lets a one-GPU box run
        # the NCCL calls, their dtypes and their stream ordering
        self.always_reduce = bool(always_reduce) and live

    def close(self):
        if hasattr(self.ops, "close"):
            self.ops.close()

    # ---- a1/a2: each rank keeps only the particles whose global address falls in its shard
    def set_j_particles(self, addr, tj, m, x, v=None, a=None, jerk=None):
        """Host arrays for particles with GLOBAL addresses addr (None: 0..n-1); every rank is given
        the same arrays and loads its own slice."""
        m = np.asarray(m)
        n = m.shape[0]
        addr = np.arange(n, dtype=np.int64) if addr is None else np.asarray(addr, dtype=np.int64)
        if addr.shape[0] != n:
            raise ValueError("set_j_particles: addr and m differ in length")
        if n and (addr.min() < 0 or addr.max() >= self.n_total):
            raise ValueError("set_j_particles: global address out of range")
        keep = np.nonzero((addr >= self.j0) & (addr < self.j1))[0]
        if keep.size == 0:
            return 0

        def cut(arr):
            return None if arr is None else np.asarray(arr)[keep]

        self.ops.set_j_local((addr[keep] - self.j0).astype(np.int32), cut(tj), m[keep], cut(x), cut(v), cut(a),
                             cut(jerk))
        return int(keep.size)

    def set_ti(self, t: float):
        self.ops.set_ti(float(t))

    def _all_reduce(self, t):
        if self.world > 1 or self.always_reduce:
            dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
            self.collectives += 1

    # ---- a4-a7 over the shards
    def calc(self, i_global, eps2: float, flags: int = B.NBK_JERK | B.NBK_POT, out=None):
        """i_global: int32 tensor [n_i] of global addresses, on the ops' device, the same on every
        rank.  Returns (acc [n_i,3], jerk [n_i,3], pot [n_i]) fp32 tensors, bit-identical on every
        rank; asynchronous on the stream for the CUDA ops.  In mode "i" without `out` the tensors are
        views of the gather buffers and stay valid until the next call."""
        n_i = int(i_global.shape[0])
        if n_i > self.ni_max:
            raise ValueError("calc: n_i > ni_max")
        if flags & B.NBK_NN:
            raise ValueError("calc: the neighbour search is not combined across shards")
        if self.mode == "i" and n_i > 0:
            return self._calc_i_sharded(i_global, n_i, float(eps2), int(flags), out)
        if out is None:
            out = (self.ops.alloc((n_i, 3), torch.float32), self.ops.alloc((n_i, 3), torch.float32),
                   self.ops.alloc((n_i,), torch.float32))
        if n_i == 0:
            return out
        il, xv, s64 = self.i_local[:n_i], self.xv[:n_i], self.sum64[:n_i]
        if hasattr(self.ops, "enter"):
            self.ops.enter()
        try:
            self.ops.gather_i(self.n_local, self.j0, n_i, i_global, il, xv)
            if self.symm is not None:   # peer memory: barrier, P2P fetch, local force, barrier, P2P combine
                self.symm.barrier(channel=0)
                self.ops.fetch_i(n_i, i_global, self.shard_begin, self.peer_base, self.xv_full)
                self.ops.calc_partial(self.n_local, n_i, il, self.xv_full, float(eps2), int(flags), s64)
                self.symm.barrier(channel=1)
                self.ops.combine(n_i, [p + self.s64_off for p in self.peer_base], *out)
                self.barriers += 2
                return out
            self._all_reduce(xv)
            self.ops.calc_partial(self.n_local, n_i, il, xv, float(eps2), int(flags), s64)
            self._all_reduce(s64)
            self.ops.finish(n_i, s64, *out)
        finally:
            if hasattr(self.ops, "leave"):
                self.ops.leave()
        return out

    # ---- i-sharding: j replicated, rank r takes rows [r c, (r+1) c) of the i-list,
    # c = ceil(n_i / G); no partial sums, one all-gather of each result array
    def _all_gather(self, full, chunk_rows):
        if self.world > 1 or self.always_reduce:
            parts = [full[r * chunk_rows:(r + 1) * chunk_rows] for r in range(self.world)]
            dist.all_gather(parts, parts[self.rank], group=self.group)
            self.collectives += 1

    def _calc_i_sharded(self, i_global, n_i, eps2, flags, out):
        c = -(-n_i // self.world)
        lo, hi = min(self.rank * c, n_i), min((self.rank + 1) * c, n_i)
        rows = c * self.world
        g_acc, g_jerk, g_pot = self.g_acc[:rows], self.g_jerk[:rows], self.g_pot[:rows]
        if hasattr(self.ops, "enter"):
            self.ops.enter()
        try:
            if hi > lo:
                sl = slice(self.rank * c, self.rank * c + (hi - lo))
                self.ops.calc_slice(self.n_total, i_global[lo:hi], eps2, flags, g_acc[sl], g_jerk[sl], g_pot[sl])
            for full in (g_acc, g_jerk, g_pot):
                self._all_gather(full, c)
            if out is None:   # views of the gather buffers: valid until the next call
                out = (g_acc[:n_i], g_jerk[:n_i], g_pot[:n_i])
            else:
                out[0].copy_(g_acc[:n_i])
                out[1].copy_(g_jerk[:n_i])
                out[2].copy_(g_pot[:n_i])
        finally:
            if hasattr(self.ops, "leave"):
                self.ops.leave()
        return out
