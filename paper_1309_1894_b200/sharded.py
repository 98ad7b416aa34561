"""Row-sharded multi-GPU apply: y = alpha*A*x + beta*y with A, x and y
split into contiguous row blocks, one per GPU, one process per GPU.

    rank g owns rows [bounds[g], bounds[g+1]) of A and of y, and the same slice of x   (square A)

Per apply (the only exchange step of the path): every rank needs the x entries its columns reference and does
not own -- its *halo*.  For a stencil in natural ordering that is a plane from each neighbour (contiguous:
sent straight out of / received straight into the x vectors, no packing); for an unstructured matrix it is
an index set per peer (packed and unpacked by the library's own gather / scatter kernels).  While the halo is in
flight the rank applies its *interior* rows (the longest run of rows that reference owned columns only) through
spmv_apply_rows; the remaining rows follow when the halo has arrived.

This module is plumbing: partition, halo and interior come from the C library (spmv_partition_rows,
spmv_external_columns), the products from spmv_apply / spmv_apply_rows, packing from spmv_gather / spmv_scatter;
the transport is torch.distributed point-to-point (NCCL over NVLink / NVSwitch on GPUs, gloo in the CPU tests of
the plumbing), or a loopback between shards held by one process (single-GPU test, 2 shards on one device).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


# ----------------------------------------------------------------------------------------------------
# host-side plan: who needs what from whom (pure index arithmetic; tested against numpy on the CPU)
# ----------------------------------------------------------------------------------------------------
@dataclass
class HaloPlan:
    rank: int
    world: int
    bounds: np.ndarray            # int64 [world + 1]
    recv_cols: list               # per peer: sorted int32 columns this rank receives from it (global indices)
    send_cols: list               # per peer: sorted int32 columns this rank sends to it (global indices)

    @staticmethod
    def contiguous(idx: np.ndarray) -> bool:
        return idx.size > 0 and int(idx[-1]) - int(idx[0]) + 1 == idx.size

    def halo_entries(self) -> int:
        return int(sum(c.size for c in self.recv_cols))


def split_by_owner(ext_cols: np.ndarray, bounds: np.ndarray, rank: int) -> list:
    """ext_cols: sorted distinct external columns of `rank` -> per-owner lists (empty for rank itself)."""
    world = bounds.size - 1
    owner = np.searchsorted(bounds, ext_cols, side="right") - 1
    assert not (owner == rank).any(), "an external column cannot be owned"
    return [np.ascontiguousarray(ext_cols[owner == q], dtype=np.int32) for q in range(world)]


def make_halo_plan(rank: int, world: int, bounds: np.ndarray, ext_cols: np.ndarray, exchange_lists) -> HaloPlan:
    """exchange_lists(recv_lists) -> send_lists: the all-to-all of the index lists (setup time, once)."""
    recv = split_by_owner(ext_cols, bounds, rank)
    send = exchange_lists(recv)
    for q, s in enumerate(send):
        assert s.size == 0 or (bounds[rank] <= s.min() and s.max() < bounds[rank + 1]), "peer asked for a column I do not own"
    return HaloPlan(rank, world, np.asarray(bounds, dtype=np.int64), recv, send)


# ----------------------------------------------------------------------------------------------------
# transports
# ----------------------------------------------------------------------------------------------------
class TorchDistTransport:
    """torch.distributed point-to-point: batch_isend_irecv (NCCL: one grouped launch over NVLink)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)

    def exchange_lists(self, recv_lists):
        out = [None] * self.world
        gathered = [None] * self.world
        self.dist.all_gather_object(gathered, [np.asarray(r) for r in recv_lists], group=self.group)
        for q in range(self.world):
            out[q] = np.ascontiguousarray(gathered[q][self.rank], dtype=np.int32)    # what q wants from me
        return out

    def start(self, sends, recvs):
        """sends / recvs: lists of (peer, tensor).  Returns a handle to wait on."""
        ops = [self.dist.P2POp(self.dist.irecv, t, p, self.group) for p, t in recvs]
        ops += [self.dist.P2POp(self.dist.isend, t, p, self.group) for p, t in sends]
        return self.dist.batch_isend_irecv(ops) if ops else []

    @staticmethod
    def wait(reqs):
        for r in reqs:
            r.wait()


class LoopbackTransport:
    """All shards live in ONE process (single-GPU test / emulation): a send is a copy into the peer's receive
    buffer, performed when both sides have posted.  Shards are stepped in lock-step by `run_lockstep`."""

    def __init__(self, world: int):
        self.world = world
        self.lists = {}
        self.posted = {}

    def view(self, rank: int):
        return _LoopbackEnd(self, rank)


class _LoopbackEnd:
    def __init__(self, hub: LoopbackTransport, rank: int):
        self.hub, self.rank, self.world = hub, rank, hub.world

    def exchange_lists(self, recv_lists):
        self.hub.lists[self.rank] = [np.asarray(r, dtype=np.int32) for r in recv_lists]
        return None                                   # resolved by ShardedSpMV.finish_setup once every end has posted

    def resolve_lists(self):
        return [self.hub.lists[q][self.rank] for q in range(self.world)]

    def start(self, sends, recvs):
        # The sender packed its buffers on ITS current stream (a shard's comm stream); the receiver copies them on
        # another stream that has no dependency on it.  An event recorded here, after the packing kernels, travels
        # with the posted sends and the receiver waits on it before it reads (without it the copy could read the
        # send buffer before the gather had written it).
        ev = None
        if any(t.is_cuda for _, t in sends):
            import torch
            ev = torch.cuda.Event()
            ev.record(torch.cuda.current_stream())
        self.hub.posted[self.rank] = (sends, recvs, ev)
        return self.rank

    def wait(self, _):
        # deliver everything addressed to me (every end has posted before anyone waits: lock-step driver)
        _, my_recvs, _ = self.hub.posted[self.rank]
        for peer, dst in my_recvs:
            peer_sends, _, peer_ev = self.hub.posted[peer]
            src = [t for p, t in peer_sends if p == self.rank]
            assert len(src) == 1 and src[0].numel() == dst.numel()
            if peer_ev is not None and dst.is_cuda:
                import torch
                torch.cuda.current_stream().wait_event(peer_ev)
            dst.copy_(src[0])


# ----------------------------------------------------------------------------------------------------
# the exchange step: x_full[halo] <- owners
# ----------------------------------------------------------------------------------------------------
class HaloExchange:
    """Moves the halo of one rank.  Contiguous index runs (stencil planes, whole slices) travel straight out of /
    into x_full; index sets are packed with `pack(idx, src, dst)` (dst[i] = src[idx[i]]) and unpacked with
    `unpack(idx, src, dst)` (dst[idx[i]] = src[i]) -- on the GPU these are the library's spmv_gather / spmv_scatter."""

    def __init__(self, plan: HaloPlan, x_full, transport, pack, unpack):
        import torch
        self.plan, self.x_full, self.t, self.pack, self.unpack = plan, x_full, transport, pack, unpack
        dev = x_full.device
        self._send, self._recv = [], []          # (peer, contiguous?, (lo, hi) | idx tensor, None | buffer)
        for q in range(plan.world):
            for cols, out in ((plan.send_cols[q], self._send), (plan.recv_cols[q], self._recv)):
                if cols.size == 0:
                    continue
                if HaloPlan.contiguous(cols):
                    out.append((q, True, (int(cols[0]), int(cols[-1]) + 1), None))
                else:
                    out.append((q, False, torch.from_numpy(np.ascontiguousarray(cols, dtype=np.int32)).to(dev),
                                torch.empty(cols.size, dtype=x_full.dtype, device=dev)))

    def bytes_received(self) -> int:
        return 8 * self.plan.halo_entries()

    def start(self):
        sends, recvs = [], []
        for q, contig, where, buf in self._send:
            if contig:
                sends.append((q, self.x_full[where[0]:where[1]]))
            else:
                self.pack(where, self.x_full, buf)
                sends.append((q, buf))
        for q, contig, where, buf in self._recv:
            recvs.append((q, self.x_full[where[0]:where[1]] if contig else buf))
        return self.t.start(sends, recvs)

    def finish(self, req):
        self.t.wait(req)
        for q, contig, where, buf in self._recv:
            if not contig:
                self.unpack(where, buf, self.x_full)


# ----------------------------------------------------------------------------------------------------
# the sharded operator
# ----------------------------------------------------------------------------------------------------
class ShardedSpMV:
    """One rank's block of rows.  `A` is the GLOBAL CSR (numpy, workloads.CSR); every rank builds the same
    matrix from the same seed and keeps its own rows (synthetic workloads: no file to scatter).

    x is held full-length on every device (x_full, 8*cols bytes): the owned slice is written by the caller through
    `x_owned`, the halo entries by the exchange, the rest is never read.  Column indices stay global, so every
    kernel family and format of the library applies unchanged to the local block (a rows_local x cols matrix)."""

    def __init__(self, A, transport, *, device="cuda:0", align: int = 512, bounds=None, tune_kw=None):
        import torch
        from . import binding
        self.torch, self.binding = torch, binding
        self.t = transport
        self.rank, self.world = transport.rank, transport.world
        self.device = torch.device(device)
        assert A.rows == A.cols, "row sharding with a conformal x partition needs a square matrix"
        self.bounds = binding.partition_rows(A.row_ptr, self.world, align) if bounds is None else np.asarray(bounds, dtype=np.int64)
        lo, hi = int(self.bounds[self.rank]), int(self.bounds[self.rank + 1])
        self.lo, self.hi, self.rows_local, self.cols = lo, hi, hi - lo, A.cols
        a, b = int(A.row_ptr[lo]), int(A.row_ptr[hi])
        rp = (A.row_ptr[lo:hi + 1].astype(np.int64) - a).astype(np.int32)
        dev = self.device
        self.S = binding.SpMV(self.rows_local, A.cols, torch.from_numpy(rp).to(dev),
                              torch.from_numpy(np.ascontiguousarray(A.col_idx[a:b])).to(dev),
                              torch.from_numpy(np.ascontiguousarray(A.val[a:b])).to(dev))
        self.nnz_local = b - a
        if tune_kw is not None:
            self.S.tune(**tune_kw)                            # (the interior split is derived after the halo plan)
        self.x_full = torch.zeros(A.cols, dtype=torch.float64, device=dev)
        self.x_owned = self.x_full[lo:hi]
        ext, self.interior = self.S.external_columns(lo, hi)
        self.ext_cols = ext
        send = transport.exchange_lists(split_by_owner(ext, self.bounds, self.rank))
        self.plan = None
        self._pending_recv = split_by_owner(ext, self.bounds, self.rank)
        if send is not None:
            self._finish(send)
        self.comm_stream = torch.cuda.Stream(device=dev) if dev.type == "cuda" else None

    def finish_setup(self):
        """Loopback only: call on every shard after all of them were constructed."""
        if self.plan is None:
            self._finish(self.t.resolve_lists())

    def _finish(self, send_lists):
        send_lists = [np.ascontiguousarray(s, dtype=np.int32) for s in send_lists]
        for s in send_lists:
            assert s.size == 0 or (self.lo <= int(s.min()) and int(s.max()) < self.hi), "peer asked for a column I do not own"
        self.plan = HaloPlan(self.rank, self.world, self.bounds, self._pending_recv, send_lists)
        # packing / unpacking run in the library's kernels: there is no torch-indexing fallback
        self.halo = HaloExchange(self.plan, self.x_full, self.t, self.binding.gather, self.binding.scatter)
        self._recompute_split()

    def _recompute_split(self):
        """Interior rows on the selected variant's range alignment; worth a separate launch only when they are
        most of the block (and the variant has a row-range form at all)."""
        al = self.S.range_align()
        ia, ib = self.interior
        if al > 0:
            ia = -(-ia // al) * al
            ib = ib if ib == self.rows_local else ib // al * al
        ok = al > 0 and self.world > 1 and ib - ia >= self.rows_local // 2 and self.plan.halo_entries() > 0
        self.split = (ia, ib) if ok else None

    def select(self, desc: str):
        self.S.select(desc)
        self._recompute_split()

    def tune(self, **kw):
        rep = self.S.tune(**kw)
        self._recompute_split()
        return rep

    # ---- y_local = alpha * A_local * x + beta * y_local   (x_owned must hold this rank's slice of x)
    def apply(self, alpha, beta, y_local):
        req = self.apply_begin(alpha, beta, y_local)
        self.apply_end(req, alpha, beta, y_local)
        return y_local

    def apply_begin(self, alpha, beta, y_local):
        torch = self.torch
        if not self.halo._send and not self.halo._recv:               # nothing to exchange (one rank, block diagonal)
            return None
        if self.comm_stream is not None:
            # the exchange runs on its own stream, after whatever produced x_owned on the current stream
            self.comm_stream.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(self.comm_stream):
                req = self.halo.start()
        else:
            req = self.halo.start()
        if self.split is not None:                                    # interior rows while the halo is in flight
            self.S.apply_rows(alpha, self.x_full, beta, y_local, self.split[0], self.split[1])
        return req

    def apply_end(self, req, alpha, beta, y_local):
        torch = self.torch
        if not self.halo._send and not self.halo._recv:
            self.S.apply(alpha, self.x_full, beta, y_local)
            return
        if self.comm_stream is not None:
            with torch.cuda.stream(self.comm_stream):
                self.halo.finish(req)
            torch.cuda.current_stream().wait_stream(self.comm_stream)
        else:
            self.halo.finish(req)
        if self.split is None:
            self.S.apply(alpha, self.x_full, beta, y_local)
        else:
            ia, ib = self.split
            if ia > 0:
                self.S.apply_rows(alpha, self.x_full, beta, y_local, 0, ia)
            if ib < self.rows_local:
                self.S.apply_rows(alpha, self.x_full, beta, y_local, ib, self.rows_local)

    def close(self):
        self.S.close()


def run_lockstep(shards, alpha, beta, ys):
    """Loopback driver: every shard posts its exchange (and applies its interior), then every shard completes."""
    reqs = [s.apply_begin(alpha, beta, y) for s, y in zip(shards, ys)]
    for s, r, y in zip(shards, reqs, ys):
        s.apply_end(r, alpha, beta, y)
