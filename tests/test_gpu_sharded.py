"""GPU tests of the row-sharded apply.  One GPU is available, so the ranks are
emulated the supported way: all shards live in ONE process and exchange through the loopback transport (copies
between the shards' buffers); nothing waits on another launch.  Products, range launches, pack and unpack run in
the library's kernels; the concatenated result is compared with oracle/ on every row."""
import numpy as np
import pytest

import oracle
from paper_1309_1894_b200 import binding, sharded
from paper_1309_1894_b200 import workloads as W
from tests import helpers as H

pytestmark = pytest.mark.gpu


def _external_columns_numpy(A, lo, hi):
    a, b = int(A.row_ptr[lo]), int(A.row_ptr[hi])
    c = A.col_idx[a:b]
    return np.unique(c[(c < lo) | (c >= hi)]).astype(np.int32)


@pytest.mark.parametrize("name,world,variant", [
    ("stencil7", 2, "dia_const:b256:r1:x0"), ("stencil7", 3, "dia_tma:b288:c256:r1:u7:i3:x0"),
    ("stencil27", 2, "sell_tma:b288:c256:s1:r1:u8:i3:x0"), ("fem", 2, "bcsr3:b256:w8:u2:x0"),
    ("powerlaw", 2, "merge:b256:i7:x0"), ("powerlaw", 4, "csr_vector:b256:w8:u2:x0"), ("banded", 2, "sell16:b256:c128:s1:r2:u4:x0"),
])
def test_sharded_apply_matches_oracle(cuda, name, world, variant):
    import torch
    A = {"stencil7": lambda: W.laplace3d_7pt(40), "stencil27": lambda: W.stencil3d_27pt(30, perturb_stream=50),
         "fem": lambda: W.fem_block27(14), "powerlaw": lambda: W.powerlaw(40000, lmax=2000),
         "banded": lambda: W.banded_random(60000, 10, 700, stream=86)}[name]()
    x, y0 = W.uniform(87, A.cols), W.uniform(88, A.rows)
    hub = sharded.LoopbackTransport(world)
    align = 768 if name == "fem" else 512                     # a multiple of 3 for the block format
    shards = [sharded.ShardedSpMV(A, hub.view(r), align=align) for r in range(world)]
    for s in shards:
        s.finish_setup()
    bounds = shards[0].bounds
    assert bounds[0] == 0 and bounds[-1] == A.rows
    n_split = 0
    for s in shards:
        # the library's halo (device kernel) equals the numpy re-derivation; interior rows reference owned columns only
        assert np.array_equal(s.ext_cols, _external_columns_numpy(A, s.lo, s.hi))
        ia, ib = s.interior
        if ib > ia:
            a, b = int(A.row_ptr[s.lo + ia]), int(A.row_ptr[s.lo + ib])
            c = A.col_idx[a:b]
            assert ((c >= s.lo) & (c < s.hi)).all()
        s.select(variant)                                      # also re-derives the interior split for this variant
        n_split += s.split is not None
        s.x_owned.copy_(torch.from_numpy(x[s.lo:s.hi]))
    if name in ("stencil7", "stencil27", "fem", "banded") and variant.split(":")[0] != "merge":
        assert n_split == world                                # banded: interior rows overlap the exchange
    for alpha, beta in ((1.0, 0.0), (-1.5, 0.5)):
        if beta != 0.0:                                        # a NEW x for the second pass: halo buffers that still hold
            x = W.uniform(91, A.cols)                          # the first pass's entries would now give a wrong result
            for s in shards:
                s.x_owned.copy_(torch.from_numpy(x[s.lo:s.hi]))
        ys = [H.to_dev(y0[s.lo:s.hi]).clone() if beta != 0.0 else
              torch.full((s.rows_local,), float("nan"), dtype=torch.float64, device="cuda") for s in shards]
        sharded.run_lockstep(shards, alpha, beta, ys)
        torch.cuda.synchronize()
        y = np.concatenate([t.cpu().numpy() for t in ys])
        y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, alpha, x, beta, None if beta == 0.0 else y0)
        ok, mr, ff, nf = oracle.accept(y, y_ref, scale, H.TOL)
        assert ok, (name, world, variant, alpha, beta, nf, ff, mr)
    # stencil halos are contiguous planes (no packing); the power-law halo is an index set
    kinds = {c for s in shards for (_, c, _, _) in s.halo._recv}
    assert kinds == ({True} if name.startswith("stencil") else kinds)
    if name == "powerlaw":
        assert False in kinds
    for s in shards:
        s.close()


def test_apply_rows_refuses_what_has_no_range_form(cuda):
    import torch
    A = W.csr_from_lengths(np.random.default_rng(5).integers(1, 20, 5000), 5000, 90)
    S = binding.SpMV.from_csr(A)
    x = H.to_dev(W.uniform(89, A.cols)); y = torch.zeros(A.rows, dtype=torch.float64, device="cuda")
    S.select("merge:b256:i7:x0")
    assert S.range_align() == 0
    with pytest.raises(binding.SpmvError) as e:
        S.apply_rows(1.0, x, 0.0, y, 0, 128)
    assert e.value.status == 3
    S.select("sell:b256:c128:s512:r1:u2:x0")
    assert S.range_align() == 512
    with pytest.raises(binding.SpmvError) as e:               # not on the alignment
        S.apply_rows(1.0, x, 0.0, y, 128, 1024)
    assert e.value.status == 3
    S.apply_rows(1.0, x, 0.0, y, 512, 1024)
    torch.cuda.synchronize()
    y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.0, x.cpu().numpy(), 0.0)
    got = y.cpu().numpy()
    assert oracle.accept(got[512:1024], y_ref[512:1024], scale[512:1024], H.TOL)[0]
    assert (got[:512] == 0).all() and (got[1024:] == 0).all()              # nothing outside the range is written
    # dia_const: the pair-load instantiation (r2) falls back to one row per thread on unaligned vectors, range form too
    L = W.laplace3d_7pt(24)
    T = binding.SpMV.from_csr(L)
    T.select("dia_const:b256:r2:x0")
    xs = W.uniform(91, L.cols)
    buf_x = torch.zeros(L.cols + 1, dtype=torch.float64, device="cuda"); buf_x[1:] = H.to_dev(xs)
    buf_y = torch.zeros(L.rows + 1, dtype=torch.float64, device="cuda")
    al = T.range_align()
    a, b = 3 * al, 9 * al
    T.apply_rows(2.0, buf_x[1:], 0.0, buf_y[1:], a, b)          # 8-byte aligned only
    torch.cuda.synchronize()
    y_ref, scale = oracle.spmv(L.row_ptr, L.col_idx, L.val, 2.0, xs, 0.0)
    got = buf_y[1:].cpu().numpy()
    assert oracle.accept(got[a:b], y_ref[a:b], scale[a:b], H.TOL)[0]
    assert (got[:a] == 0).all() and (got[b:] == 0).all()
    T.close()
    S.close()


def test_torch_distributed_transport_world1_nccl(cuda):
    """The production transport (torch.distributed over NCCL) with the one rank this box has: process-group set-up,
    the setup-time list exchange, an apply without peers.  (More ranks need more GPUs; the exchange itself is
    covered by the gloo world-2 test on the CPU and by the loopback shards above.)"""
    import os
    import socket
    import torch
    import torch.distributed as dist
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda:0"))
    try:
        A = W.laplace3d_7pt(30)
        sh = sharded.ShardedSpMV(A, sharded.TorchDistTransport(), device="cuda:0")
        assert sh.plan is not None and sh.plan.halo_entries() == 0 and sh.split is None
        assert list(sh.bounds) == [0, A.rows]
        x, y0 = W.uniform(92, A.cols), W.uniform(93, A.rows)
        sh.x_owned.copy_(H.to_dev(x))
        y = H.to_dev(y0).clone()
        sh.apply(1.5, -0.5, y)
        torch.cuda.synchronize()
        y_ref, scale = oracle.spmv(A.row_ptr, A.col_idx, A.val, 1.5, x, -0.5, y0)
        assert oracle.accept(y.cpu().numpy(), y_ref, scale, H.TOL)[0]
        sh.close()
    finally:
        dist.destroy_process_group()
