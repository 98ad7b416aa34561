"""Seeded synthetic inputs (numpy only) shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic: it only builds CSR matrices and
vectors.  Both the oracle (oracle/) and the CUDA library consume the arrays produced
here; neither side generates its own inputs.

Recipes follow BASELINE.json:configs and the readings of SURVEY.md sec. 8(c)/(d)
(A10 counter-based RNG, A11 truncated Zipf, A12 Dirichlet truncation + lexicographic
ordering, A13 config 4 built by structure, A14 diagonal shift on the global diagonal,
A15 alpha/beta defaults, A16 per-entry perturbations).  They stand in for the
"stencil-based computations" of the paper's refs [1],[2]; the paper
names no dataset.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

_U64 = np.uint64
_CHUNK = 1 << 24


# ----------------------------------------------------------------------------
# counter-based RNG (reading A10): splitmix64 finaliser on (stream, index)
# ----------------------------------------------------------------------------
def mix64(stream: int, idx: np.ndarray) -> np.ndarray:
    """64-bit hash of (stream, idx); idx is a uint64 array of counters."""
    with np.errstate(over="ignore"):
        z = idx.astype(_U64) + _U64((0x9E3779B97F4A7C15 * (2 * stream + 1)) & 0xFFFFFFFFFFFFFFFF)
        z ^= z >> _U64(30)
        z *= _U64(0xBF58476D1CE4E5B9)
        z ^= z >> _U64(27)
        z *= _U64(0x94D049BB133111EB)
        z ^= z >> _U64(31)
        z += _U64((0xD6E8FEB86659FD93 * (stream + 1)) & 0xFFFFFFFFFFFFFFFF)
        z ^= z >> _U64(32)
        z *= _U64(0xD6E8FEB86659FD93)
        z ^= z >> _U64(32)
    return z


def _unit(stream: int, lo: int, hi: int) -> np.ndarray:
    """U[0,1) from counters lo..hi-1 (top 53 bits / 2^53)."""
    z = mix64(stream, np.arange(lo, hi, dtype=_U64))
    return (z >> _U64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def uniform(stream: int, n: int, lo: float = -1.0, hi: float = 1.0) -> np.ndarray:
    """n samples of U[lo,hi) from counter stream `stream`."""
    out = np.empty(n, dtype=np.float64)
    for a in range(0, n, _CHUNK):
        b = min(n, a + _CHUNK)
        out[a:b] = lo + (hi - lo) * _unit(stream, a, b)
    return out


def normal(stream: int, n: int) -> np.ndarray:
    """n samples of N(0,1): Box-Muller on counters (2i, 2i+1)."""
    out = np.empty(n, dtype=np.float64)
    for a in range(0, n, _CHUNK):
        b = min(n, a + _CHUNK)
        z = mix64(stream, np.arange(2 * a, 2 * b, dtype=_U64))
        u = (z >> _U64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
        u1 = 1.0 - u[0::2]          # (0,1]
        u2 = u[1::2]
        out[a:b] = np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
    return out


# ----------------------------------------------------------------------------
# CSR container
# ----------------------------------------------------------------------------
@dataclass
class CSR:
    rows: int
    cols: int
    row_ptr: np.ndarray   # int32 [rows+1]
    col_idx: np.ndarray   # int32 [nnz]
    val: np.ndarray       # float64 [nnz]

    @property
    def nnz(self) -> int:
        return int(self.row_ptr[-1])

    def row_lengths(self) -> np.ndarray:
        return np.diff(self.row_ptr)


def csr_from_lengths(lengths, cols: int, stream: int, *, sort=True, values="normal") -> CSR:
    """Random CSR with the given row lengths; distinct uniform columns per row."""
    lengths = np.asarray(lengths, dtype=np.int64)
    rows = lengths.size
    assert lengths.max(initial=0) <= cols
    row_ptr = np.zeros(rows + 1, dtype=np.int64)
    np.cumsum(lengths, out=row_ptr[1:])
    nnz = int(row_ptr[-1])
    assert nnz < 2**31
    col_idx = _distinct_columns(row_ptr, cols, stream)
    if not sort:
        # deterministic within-row shuffle: sort by a hash instead of by column
        rid = np.repeat(np.arange(rows, dtype=_U64), lengths)
        h = mix64(stream + 7, np.arange(nnz, dtype=_U64)) >> _U64(24)
        order = np.argsort((rid << _U64(40)) | h, kind="stable")
        col_idx = col_idx[order]
    if values == "normal":
        val = normal(stream + 1, nnz)
    elif values == "ones":
        val = np.ones(nnz)
    elif values == "smallint":
        val = (mix64(stream + 1, np.arange(nnz, dtype=_U64)) % _U64(17)).astype(np.float64) - 8.0
    else:
        raise ValueError(values)
    return CSR(rows, cols, row_ptr.astype(np.int32), col_idx.astype(np.int32), val)


def _distinct_columns(row_ptr: np.ndarray, cols: int, stream: int, lo=None, span=None) -> np.ndarray:
    """Per row: uniform draws from [0, cols) -- or from [lo[row], lo[row] + span[row]) when given --
    duplicates rejected and redrawn, sorted.
    (BASELINE.json:configs[2] "columns uniform random without replacement ... sorted")."""
    rows = row_ptr.size - 1
    nnz = int(row_ptr[-1])
    if nnz == 0:
        return np.zeros(0, dtype=np.int64)
    lengths = np.diff(row_ptr)
    rid = np.repeat(np.arange(rows, dtype=_U64), lengths)
    shift = _U64(32)
    key = np.empty(nnz, dtype=_U64)
    if lo is not None:
        assert (2 * lengths <= span).all(), "windowed draws need rows at most half as long as their window"
        e_lo = np.repeat(np.asarray(lo, dtype=_U64), lengths)
        e_span = np.repeat(np.asarray(span, dtype=_U64), lengths)
        draw = lambda strm, idx, sel: e_lo[sel] + mix64(strm, idx) % e_span[sel]
        key[:] = (rid << shift) | draw(stream, np.arange(nnz, dtype=_U64), slice(None))
        attempt = 0
        while True:
            key.sort()
            dup = np.flatnonzero(key[1:] == key[:-1]) + 1
            if dup.size == 0:
                break
            attempt += 1
            assert attempt < 1000, "column rejection sampling did not converge"
            # after sorting, entry `dup` still belongs to row key >> 32: redraw inside that row's window
            r = (key[dup] >> shift).astype(np.int64)
            lo_a, span_a = np.asarray(lo, dtype=_U64), np.asarray(span, dtype=_U64)
            key[dup] = (key[dup] & ~_U64(0xFFFFFFFF)) | (lo_a[r] + mix64(stream + 1000 * attempt, dup.astype(_U64)) % span_a[r])
        return (key & _U64(0xFFFFFFFF)).astype(np.int64)
    for a in range(0, nnz, _CHUNK):
        b = min(nnz, a + _CHUNK)
        key[a:b] = (rid[a:b] << shift) | (mix64(stream, np.arange(a, b, dtype=_U64)) % _U64(cols))
    # rows needing more than half of all columns (tiny test matrices only): rejection
    # would not converge, so take the `length` columns with the smallest hash instead
    for i in np.flatnonzero(2 * lengths > cols):
        h = mix64(stream + 500, np.arange(i * cols, (i + 1) * cols, dtype=_U64))
        pick = np.sort(np.argsort(h, kind="stable")[:lengths[i]]).astype(_U64)
        key[row_ptr[i]:row_ptr[i + 1]] = (_U64(i) << shift) | pick
    attempt = 0
    while True:
        key.sort()
        dup = np.flatnonzero(key[1:] == key[:-1]) + 1
        if dup.size == 0:
            break
        attempt += 1
        assert attempt < 1000, "column rejection sampling did not converge"
        c = mix64(stream + 1000 * attempt, dup.astype(_U64)) % _U64(cols)
        key[dup] = (rid[dup] << shift) | c
    return (key & _U64(0xFFFFFFFF)).astype(np.int64)


# ----------------------------------------------------------------------------
# stencil matrices (reading A12: Dirichlet truncation, row = i + n*(j + n*k))
# ----------------------------------------------------------------------------
def _stencil_padded(n: int, dim: int, offsets, lo: int = 0, hi: int | None = None):
    """Padded neighbour table for grid points lo..hi-1 of an n^dim grid: returns
    (cols int64 [M,S], mask bool [M,S], index of the centre offset).  Offsets are
    tuples of length dim (fastest index first), ordered by ascending column."""
    N = n ** dim
    hi = N if hi is None else hi
    idx = np.arange(lo, hi, dtype=np.int64)
    coords = []
    r = idx
    for _ in range(dim):
        coords.append(r % n)
        r = r // n
    strides = [n ** d for d in range(dim)]
    offs = sorted(offsets, key=lambda o: sum(o[d] * strides[d] for d in range(dim)))
    S = len(offs)
    cols = np.empty((idx.size, S), dtype=np.int64)
    mask = np.empty((idx.size, S), dtype=bool)
    for s, o in enumerate(offs):
        ok = np.ones(idx.size, dtype=bool)
        delta = 0
        for d in range(dim):
            if o[d] != 0:
                c = coords[d] + o[d]
                ok &= (c >= 0) & (c < n)
            delta += o[d] * strides[d]
        cols[:, s] = idx + delta
        mask[:, s] = ok
    return cols, mask, offs.index(tuple([0] * dim))


def _stencil_pattern(n: int, dim: int, offsets):
    """Returns (row_ptr int64, col_idx int64, is_diag bool[nnz]) (Dirichlet truncation)."""
    N = n ** dim
    step = 1 << 20
    lens, cis, dgs = [], [], []
    for a in range(0, N, step):
        cols, mask, ds = _stencil_padded(n, dim, offsets, a, min(N, a + step))
        lens.append(mask.sum(axis=1))
        cis.append(cols[mask])
        isd = np.zeros(mask.shape, dtype=bool)
        isd[:, ds] = True
        dgs.append(isd[mask])
    row_ptr = np.zeros(N + 1, dtype=np.int64)
    np.cumsum(np.concatenate(lens), out=row_ptr[1:])
    return row_ptr, np.concatenate(cis), np.concatenate(dgs)


def _finish(N, row_ptr, col_idx, val) -> CSR:
    assert int(row_ptr[-1]) < 2**31
    return CSR(N, N, row_ptr.astype(np.int32), col_idx.astype(np.int32),
               np.ascontiguousarray(val, dtype=np.float64))


def laplace2d_5pt(n: int, diag: float = 4.0, off: float = -1.0) -> CSR:
    offs = [(0, 0), (1, 0), (-1, 0), (0, 1), (0, -1)]
    rp, ci, dg = _stencil_pattern(n, 2, offs)
    return _finish(n * n, rp, ci, np.where(dg, diag, off))


def laplace3d_7pt(n: int, diag: float = 6.0, off: float = -1.0) -> CSR:
    offs = [(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)]
    rp, ci, dg = _stencil_pattern(n, 3, offs)
    return _finish(n ** 3, rp, ci, np.where(dg, diag, off))


def _offs27():
    return [(a, b, c) for c in (-1, 0, 1) for b in (-1, 0, 1) for a in (-1, 0, 1)]


def stencil3d_27pt(n: int, diag: float = 26.0, off: float = -1.0,
                   perturb_stream: int | None = None, perturb: float = 0.01) -> CSR:
    rp, ci, dg = _stencil_pattern(n, 3, _offs27())
    val = np.where(dg, diag, off).astype(np.float64)
    if perturb_stream is not None:          # reading A16: every stored entry perturbed
        val += uniform(perturb_stream, val.size, -perturb, perturb)
    return _finish(n ** 3, rp, ci, val)


def fem_block27(n: int, dof: int = 3, val_stream: int = 40, shift: float = 30.0) -> CSR:
    """27-point connectivity on n^3 nodes, dense dof x dof blocks (readings A13, A14):
    scalar row = dof*node + d; every scalar entry ~ N(0,1) from (val_stream, k), k the
    CSR position; +shift on the global diagonal."""
    Nn = n ** 3
    rows = Nn * dof
    e = np.arange(dof, dtype=np.int64)
    step = 1 << 17
    lens, cis = [], []
    for a in range(0, Nn, step):
        cols, mask, _ = _stencil_padded(n, 3, _offs27(), a, min(Nn, a + step))
        M, S = cols.shape
        sc = (cols[:, :, None] * dof + e[None, None, :]).reshape(M, S * dof)
        sm = np.repeat(mask, dof, axis=1)
        sc = np.repeat(sc, dof, axis=0)          # the dof scalar rows of a node share a column list
        sm = np.repeat(sm, dof, axis=0)
        lens.append(sm.sum(axis=1))
        cis.append(sc[sm].astype(np.int32))
    lengths = np.concatenate(lens)
    row_ptr = np.zeros(rows + 1, dtype=np.int64)
    np.cumsum(lengths, out=row_ptr[1:])
    nnz = int(row_ptr[-1])
    assert nnz < 2**31
    col_idx = np.concatenate(cis)
    del cis
    val = normal(val_stream, nnz)
    for a in range(0, rows, 1 << 20):            # +shift where col == row
        b = min(rows, a + (1 << 20))
        rid = np.repeat(np.arange(a, b, dtype=np.int32), lengths[a:b])
        seg = slice(int(row_ptr[a]), int(row_ptr[b]))
        val[seg][col_idx[seg] == rid] += shift
    return CSR(rows, rows, row_ptr.astype(np.int32), col_idx, val)


# ----------------------------------------------------------------------------
# power-law matrix (reading A11: truncated, renormalised Zipf)
# ----------------------------------------------------------------------------
def zipf_lengths(rows: int, s: float = 1.8, lmax: int = 20000, stream: int = 30) -> np.ndarray:
    k = np.arange(1, lmax + 1, dtype=np.float64)
    pmf = k ** (-s)
    cdf = np.cumsum(pmf / pmf.sum())
    u = uniform(stream, rows, 0.0, 1.0)
    L = np.searchsorted(cdf, u, side="right") + 1
    return np.minimum(L, lmax).astype(np.int64)


def powerlaw(rows: int, cols: int | None = None, s: float = 1.8, lmax: int = 20000,
             len_stream: int = 30, col_stream: int = 31, val_stream: int = 32) -> CSR:
    cols = rows if cols is None else cols
    lengths = zipf_lengths(rows, s, min(lmax, cols), len_stream)
    row_ptr = np.zeros(rows + 1, dtype=np.int64)
    np.cumsum(lengths, out=row_ptr[1:])
    nnz = int(row_ptr[-1])
    assert nnz < 2**31
    col_idx = _distinct_columns(row_ptr, cols, col_stream)
    val = normal(val_stream, nnz)
    return CSR(rows, cols, row_ptr.astype(np.int32), col_idx.astype(np.int32), val)


def banded_random(rows: int, per_row: int = 24, half_band: int = 12000, stream: int = 80) -> CSR:
    """Square banded matrix with UNSTRUCTURED columns inside the band (a finite-element matrix on an
    irregular mesh after bandwidth-reducing reordering): every row holds `per_row` distinct columns drawn
    uniformly from [i - half_band, i + half_band] (clipped to the matrix), sorted; values N(0,1).
    Thousands of distinct diagonals, so the DIA family refuses it, while every SELL slice spans fewer than
    65535 columns: the workload of the 16-bit delta-index variants."""
    i = np.arange(rows, dtype=np.int64)
    lo = np.maximum(i - half_band, 0)
    hi = np.minimum(i + half_band, rows - 1)
    span = hi - lo + 1
    lengths = np.minimum(per_row, span // 2).astype(np.int64)
    row_ptr = np.zeros(rows + 1, dtype=np.int64)
    np.cumsum(lengths, out=row_ptr[1:])
    col_idx = _distinct_columns(row_ptr, rows, stream, lo=lo, span=span)
    return CSR(rows, rows, row_ptr.astype(np.int32), col_idx.astype(np.int32), normal(stream + 1, int(row_ptr[-1])))


# ----------------------------------------------------------------------------
# the five BASELINE.json configs
# ----------------------------------------------------------------------------
@dataclass
class Problem:
    name: str
    A: CSR
    x: np.ndarray
    y0: np.ndarray | None
    alpha: float
    beta: float
    note: str = ""
    extra: dict = field(default_factory=dict)


CONFIG_NAMES = {
    1: "cfg1: 2D 5-pt Laplacian 64^2 (Dirichlet), alpha=1 beta=0",
    2: "cfg2: 3D 7-pt Laplacian 128^3, alpha=1 beta=0.5",
    3: "cfg3: power-law Zipf(1.8) on [1,20000], 4194304^2, alpha=1 beta=0",
    4: "cfg4: FEM 27-pt x 3x3 blocks, 96^3 nodes, alpha=1 beta=0",
    5: "cfg5: 4 x 3D 27-pt 128^3 perturbed, alpha=1 beta=1",
}


def config(cfg: int, scale: float = 1.0, member: int = 0) -> Problem:
    """Problem for BASELINE.json:configs[cfg-1].  `scale` < 1 shrinks the grid / row
    count (same recipe, same seeds) for tests; `member` selects the matrix of cfg 5."""
    if cfg == 1:
        n = max(2, int(round(64 * scale)))
        A = laplace2d_5pt(n)
        return Problem(CONFIG_NAMES[1], A, uniform(0, A.cols), None, 1.0, 0.0)
    if cfg == 2:
        n = max(2, int(round(128 * scale)))
        A = laplace3d_7pt(n)
        return Problem(CONFIG_NAMES[2], A, uniform(20, A.cols), uniform(21, A.rows), 1.0, 0.5)
    if cfg == 3:
        rows = max(64, int(round(4194304 * scale)))
        A = powerlaw(rows)
        return Problem(CONFIG_NAMES[3], A, uniform(33, A.cols), None, 1.0, 0.0)
    if cfg == 4:
        n = max(2, int(round(96 * scale)))
        A = fem_block27(n)
        return Problem(CONFIG_NAMES[4], A, uniform(41, A.cols), None, 1.0, 0.0,
                       note="BASELINE.json says ~71M nnz; structure gives 9*(3n-2)^3 (SURVEY A13)")
    if cfg == 5:
        n = max(2, int(round(128 * scale)))
        m = member
        A = stencil3d_27pt(n, 26.0, -1.0, perturb_stream=50 + m)
        return Problem(CONFIG_NAMES[5] + f" [matrix {m}]", A, uniform(54 + m, A.cols),
                       uniform(58 + m, A.rows), 1.0, 1.0)
    raise ValueError(cfg)


def algorithmic_bytes(rows: int, cols: int, nnz: int, beta: float) -> int:
    """Byte model of BASELINE.json:north_star / SURVEY 8(d):
    nnz*(8+4) + (rows+1)*4 + 8*cols (x) + 8*rows (y write) [+ 8*rows if beta != 0]."""
    return nnz * 12 + (rows + 1) * 4 + 8 * cols + 8 * rows + (8 * rows if beta != 0.0 else 0)
