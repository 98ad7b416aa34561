"""CPU tests of the row-sharded apply's host side: the nnz-balanced partition
(spmv_partition_rows: plain host code in the C library), the halo index sets, and -- with two gloo processes --
the exchange itself.  The kernels (products, pack / unpack) are GPU-only and tested in test_gpu_sharded.py; here
pack / unpack are numpy stand-ins supplied BY THE TEST (the product has no such fallback)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1309_1894_b200 import binding, sharded
from paper_1309_1894_b200 import workloads as W


def _external_columns_numpy(A, lo, hi):
    a, b = int(A.row_ptr[lo]), int(A.row_ptr[hi])
    c = A.col_idx[a:b]
    return np.unique(c[(c < lo) | (c >= hi)]).astype(np.int32)


def test_partition_is_nnz_balanced_aligned_and_monotone():
    for A, parts, align in ((W.powerlaw(30000, lmax=3000), 8, 128), (W.laplace3d_7pt(20), 4, 512),
                            (W.csr_from_lengths([0] * 50 + [7] * 50, 80, 3), 3, 1), (W.laplace2d_5pt(8), 5, 16)):
        b = binding.partition_rows(A.row_ptr, parts, align)
        assert b[0] == 0 and b[-1] == A.rows and (np.diff(b) >= 0).all()
        assert all(int(v) % align == 0 for v in b[1:-1])
        # numpy re-derivation: first row whose prefix count reaches g*nnz/parts, rounded to the alignment
        for g in range(1, parts):
            r = int(np.searchsorted(A.row_ptr, A.nnz * g // parts, side="left"))
            r = min((r + align // 2) // align * align, A.rows)
            assert b[g] == max(r, b[g - 1])
        if A.rows >= 100 * parts * align:                     # balance, where the alignment leaves room for it
            per = np.diff(A.row_ptr[b].astype(np.int64))
            assert per.max() <= 1.1 * A.nnz / parts + A.row_lengths().max() * align


def test_halo_sets_of_a_stencil_are_planes_and_of_a_random_matrix_are_index_lists():
    n = 12
    A = W.laplace3d_7pt(n)
    bounds = binding.partition_rows(A.row_ptr, 3, n * n)
    lists = {}
    for r in range(3):
        lo, hi = int(bounds[r]), int(bounds[r + 1])
        ext = _external_columns_numpy(A, lo, hi)
        recv = sharded.split_by_owner(ext, bounds, r)
        lists[r] = recv
        for q in range(3):
            if abs(q - r) == 1:                               # exactly the neighbouring plane, contiguous
                plane = np.arange(lo - n * n, lo) if q < r else np.arange(hi, hi + n * n)
                assert np.array_equal(recv[q], plane) and sharded.HaloPlan.contiguous(recv[q])
            else:
                assert recv[q].size == 0
    # what q receives from r is what r sends to q
    send_0_to_1 = lists[1][0]
    assert np.array_equal(send_0_to_1, np.arange(bounds[1] - n * n, bounds[1]))
    B = W.powerlaw(5000, lmax=400)
    bb = binding.partition_rows(B.row_ptr, 4, 64)
    for r in range(4):
        ext = _external_columns_numpy(B, int(bb[r]), int(bb[r + 1]))
        recv = sharded.split_by_owner(ext, bb, r)
        assert recv[r].size == 0 and sum(x.size for x in recv) == ext.size
        for q in range(4):
            assert ((recv[q] >= bb[q]) & (recv[q] < bb[q + 1])).all() and (np.diff(recv[q]) > 0).all()


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    t = sharded.TorchDistTransport()
    out = {}
    for name, A in (("stencil", W.laplace3d_7pt(10)), ("random", W.powerlaw(3000, lmax=300))):
        bounds = binding.partition_rows(A.row_ptr, world, 4)
        lo, hi = int(bounds[rank]), int(bounds[rank + 1])
        ext = _external_columns_numpy(A, lo, hi)
        plan = sharded.make_halo_plan(rank, world, bounds, ext, t.exchange_lists)
        x = W.uniform(7, A.cols)
        x_full = torch.zeros(A.cols, dtype=torch.float64)
        x_full[lo:hi] = torch.from_numpy(x[lo:hi])
        ex = sharded.HaloExchange(plan, x_full, t,
                                  pack=lambda idx, src, dst: dst.copy_(src[idx.long()]),
                                  unpack=lambda idx, src, dst: dst.index_copy_(0, idx.long(), src))
        ex.finish(ex.start())
        got = x_full.numpy()
        need = np.concatenate([np.arange(lo, hi), ext])
        out[name] = (bool(np.array_equal(got[need], x[need])), int(ext.size), ex.bytes_received(),
                     [bool(sharded.HaloPlan.contiguous(c)) for c in plan.recv_cols if c.size])
    q.put((rank, out))
    dist.barrier()
    dist.destroy_process_group()


def test_halo_exchange_gloo_world2():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    got = dict(q.get(timeout=180) for _ in range(2))
    for p in ps:
        p.join(180)
        assert p.exitcode == 0
    for rank in (0, 1):
        ok, n_ext, nbytes, contig = got[rank]["stencil"]
        assert ok and n_ext == 100 and nbytes == 800 and contig == [True]        # one 10x10 plane from the neighbour
        ok, n_ext, nbytes, contig = got[rank]["random"]
        assert ok and n_ext > 100 and nbytes == 8 * n_ext and contig == [False]   # an index set: packed / unpacked
