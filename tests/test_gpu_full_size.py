"""GPU parity at BASELINE.json's full sizes (-m gpu), in the launch configuration bench.py times:
one Context, device-resident inputs, one sdp_align_batch call per config on the full pair list.

Every config is compared with the oracle on EVERY pair, in the default mode and in SDP_MODE_LOCAL (the oracle
needs about two minutes per mode for the four configs on 16 host cores), and properties that hold at any size are checked on all pairs as well (score
bounds, CIGAR consumes the read and the reported window span, offsets are the exclusive scan of the
lengths). `sample` stays as a knob for quick local runs."""
import os

import numpy as np
import pytest

from oracle import OracleScoring
from paper_1302_5507_b200 import Context, workloads as W

import parity

pytestmark = pytest.mark.gpu
DEFAULT = OracleScoring(1, -3, 5, 2, 0.6)
FULL = os.environ.get("SDP_FULL_SIZE_TESTS", "1") != "0"


def cigar_spans(got):
    """(read bases, window bases, runs) consumed per pair, from the compacted CIGAR buffer."""
    ops = got.cigar_ops.astype(np.int64)
    length, op = ops >> 4, ops & 15
    seg = np.repeat(np.arange(len(got.cigar_len)), got.cigar_len.astype(np.int64))
    read_b = np.bincount(seg, weights=length * (op != 2), minlength=len(got.cigar_len)).astype(np.int64)
    win_b = np.bincount(seg, weights=length * (op != 1), minlength=len(got.cigar_len)).astype(np.int64)
    cols = np.bincount(seg, weights=length, minlength=len(got.cigar_len)).astype(np.int64)
    return read_b, win_b, cols


def check_properties_local(batch, got, sc):
    """SDP_MODE_LOCAL (sdp.h, R18): soft clips (op 4) complete the read, aligned columns exclude them."""
    n = batch.read_len[batch.pairs[:, 0]].astype(np.int64)
    m = batch.win_len[batch.pairs[:, 1]].astype(np.int64)
    assert np.all(got.score >= 0) and np.all(got.score <= n * sc.match)
    empty = got.score == 0
    assert np.all(got.ref_end[empty] == -1) and np.all(got.read_end[empty] == -1) and not got.passed[empty].any()
    assert np.all((got.ref_end[~empty] >= 0) & (got.ref_end[~empty] < m[~empty])) and np.all(got.ref_start >= 0)
    assert np.all((got.read_start >= 0) & (got.read_end < n))
    ops = got.cigar_ops.astype(np.int64)
    length, op = ops >> 4, ops & 15
    seg = np.repeat(np.arange(len(got.cigar_len)), got.cigar_len.astype(np.int64))
    P = len(got.cigar_len)
    read_b = np.bincount(seg, weights=length * (op != 2), minlength=P).astype(np.int64)
    aligned_read = np.bincount(seg, weights=length * ((op == 0) | (op == 1)), minlength=P).astype(np.int64)
    win_b = np.bincount(seg, weights=length * ((op == 0) | (op == 2)), minlength=P).astype(np.int64)
    cols = np.bincount(seg, weights=length * (op != 4), minlength=P).astype(np.int64)
    assert np.array_equal(read_b, n)
    assert np.array_equal(aligned_read, got.read_end.astype(np.int64) - got.read_start + 1)
    assert np.array_equal(win_b, got.ref_end.astype(np.int64) - got.ref_start + 1)
    assert np.array_equal(cols, got.n_cols.astype(np.int64))
    off = np.concatenate([[0], np.cumsum(got.cigar_len.astype(np.int64))])
    assert np.array_equal(off[:-1], got.cigar_off.astype(np.int64)) and off[-1] == len(got.cigar_ops)
    q = int(round(sc.min_similarity * 1e6))
    ncols = got.n_cols.astype(np.int64)
    assert np.array_equal(got.passed.astype(bool),
                          (ncols > 0) & (got.n_match.astype(np.int64) * 1000000 >= q * (ncols + n - aligned_read)))


def check_properties(batch, got, sc):
    n = batch.read_len[batch.pairs[:, 0]].astype(np.int64)
    m = batch.win_len[batch.pairs[:, 1]].astype(np.int64)
    assert np.all(got.score <= n * sc.match) and np.all(got.score >= -(sc.gap_open + sc.gap_extend * n))
    assert np.all((got.ref_end >= 0) & (got.ref_end < m)) and np.all(got.ref_start >= 0)
    assert np.all(got.read_start == 0) and np.all(got.read_end == n - 1)
    read_b, win_b, cols = cigar_spans(got)
    assert np.array_equal(read_b, n)
    assert np.array_equal(win_b, got.ref_end.astype(np.int64) - got.ref_start + 1)
    assert np.array_equal(cols, got.n_cols.astype(np.int64))
    assert np.all(got.n_match <= got.n_cols)
    off = np.concatenate([[0], np.cumsum(got.cigar_len.astype(np.int64))])
    assert np.array_equal(off[:-1], got.cigar_off.astype(np.int64)) and off[-1] == len(got.cigar_ops)
    q = int(round(sc.min_similarity * 1e6))
    assert np.array_equal(got.passed.astype(bool), got.n_match.astype(np.int64) * 1000000 >= q * got.n_cols.astype(np.int64))


def compare_sample(batch, got, idx, sc, what, local=False):
    sub = batch.subset(idx)
    exp = parity.run_oracle(sub, sc, local=local)
    for f in ("score", "ref_end", "ref_start", "read_start", "read_end", "n_match", "n_cols", "passed", "cigar_len"):
        a, b = getattr(exp, f).astype(np.int64), getattr(got, f)[idx].astype(np.int64)
        bad = np.nonzero(a != b)[0]
        assert len(bad) == 0, f"{what}: {len(bad)} sampled pairs differ in {f}; first is pair {int(idx[bad[0]])}"
    # CIGAR runs of the sampled pairs, gathered from the compacted buffer
    lens = got.cigar_len[idx].astype(np.int64)
    starts = got.cigar_off[idx].astype(np.int64)
    take = np.repeat(starts - np.concatenate([[0], np.cumsum(lens)[:-1]]), lens) + np.arange(int(lens.sum()))
    assert np.array_equal(got.cigar_ops[take], exp.cigar_ops), f"{what}: CIGAR runs differ on the sample"


@pytest.mark.skipif(not FULL, reason="SDP_FULL_SIZE_TESTS=0")
@pytest.mark.parametrize("local", [False, True], ids=["semiglobal", "local"])
@pytest.mark.parametrize("cfg,sample", [(2, None), (3, None), (4, None), (5, None)])
def test_full_size_config(cfg, sample, local):
    batch = W.make_config(cfg)
    with Context(DEFAULT.match, DEFAULT.mismatch, DEFAULT.gap_open, DEFAULT.gap_extend, DEFAULT.min_similarity,
                 device=0) as ctx:
        ctx.set_mode(local=local)                      # local: SURVEY.md 8(f2), every pair on the int32 lane
        got = ctx.fetch(ctx.align_batch(ctx.upload(batch)))
        stats = ctx.stats()
    assert stats["cells_forward"] == batch.cells
    (check_properties_local if local else check_properties)(batch, got, DEFAULT)
    if sample is None:
        idx = np.arange(batch.n_pairs)
    else:
        idx = np.sort(np.random.default_rng(1302_5507 + cfg).choice(batch.n_pairs, size=sample, replace=False))
    compare_sample(batch, got, idx, DEFAULT, f"cfg{cfg} full size{' (local)' if local else ''}", local=local)
