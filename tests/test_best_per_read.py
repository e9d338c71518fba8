"""many candidate windows per read and the per-read choice among them.

CPU part: pins oracle.best_per_read (a sequential scan) against an independently written lexicographic sort and
hand-made cases. GPU part: sdp_best_per_read against the oracle on a step-3 shaped batch."""
import numpy as np
import pytest

import oracle
from oracle import OracleScoring
from paper_1302_5507_b200 import workloads as W

INT_MIN = -(2 ** 31)


def by_sorting(pairs, score, n_reads):
    """Independent restatement: sort each read's pairs by (-score, window, pair index) and read off ranks 0 and 1."""
    out = dict(best_pair=np.full(n_reads, 0xFFFFFFFF, np.uint32), best_score=np.full(n_reads, INT_MIN, np.int32),
               second_score=np.full(n_reads, INT_MIN, np.int32), n_candidates=np.zeros(n_reads, np.uint32))
    for r in range(n_reads):
        mine = [p for p in range(len(pairs)) if pairs[p][0] == r]
        mine.sort(key=lambda p: (-int(score[p]), int(pairs[p][1]), p))
        out["n_candidates"][r] = len(mine)
        if mine:
            out["best_pair"][r], out["best_score"][r] = mine[0], score[mine[0]]
        if len(mine) > 1:
            out["second_score"][r] = score[mine[1]]
    return out


def test_hand_made_cases():
    pairs = np.array([[0, 5], [0, 2], [0, 9], [2, 1], [2, 1], [3, 7]], dtype=np.uint32)
    score = np.array([10, 10, 3, -4, -4, 0], dtype=np.int32)
    got = oracle.best_per_read(pairs, score, 5)
    assert list(got["best_pair"]) == [1, 0xFFFFFFFF, 3, 5, 0xFFFFFFFF]      # tie on score -> lower window; equal pairs -> first
    assert list(got["best_score"][[0, 2, 3]]) == [10, -4, 0]
    assert list(got["second_score"]) == [10, INT_MIN, -4, INT_MIN, INT_MIN]
    assert list(got["n_candidates"]) == [3, 0, 2, 1, 0]


def test_oracle_scan_equals_sorting_definition():
    rng = np.random.default_rng(5)
    for _ in range(60):
        n_reads, P = int(rng.integers(1, 12)), int(rng.integers(0, 60))
        pairs = np.stack([rng.integers(0, n_reads, P), rng.integers(0, 6, P)], axis=1).astype(np.uint32)
        score = rng.integers(-5, 6, P).astype(np.int32)                    # few distinct values: many ties
        a, b = oracle.best_per_read(pairs, score, n_reads), by_sorting(pairs, score, n_reads)
        for k in a:
            assert np.array_equal(a[k], b[k]), k


def test_step3_workload_shape():
    b = W.make_step3(200, max_candidates=30, ref_bases=500_000)
    counts = np.bincount(b.pairs[:, 0], minlength=200)
    assert counts.min() >= 1 and counts.max() <= 30 and b.n_pairs == counts.sum()
    assert np.all(np.diff(b.pairs[:, 0].astype(np.int64)) >= 0)            # grouped by read
    assert int(b.win_off.max()) + int(b.win_len[0]) <= b.wins_packed.shape[0] * 16


def test_long_read_workload_shape():
    # bench.py's local / int32_lane blocks: config 2's recipe at other lengths, seeded and reproducible
    a = W.make_long_reads(40, 600, 2000, ref_bases=400_000)
    b = W.make_long_reads(40, 600, 2000, ref_bases=400_000)
    assert a.n_pairs == 40 and (a.read_len == 600).all() and (a.win_len == 2000).all() and a.cells == 40 * 600 * 2000
    assert np.array_equal(a.reads_packed, b.reads_packed) and np.array_equal(a.win_off, b.win_off)
    assert int(a.win_off.max()) + 2000 <= a.wins_packed.shape[0] * 16
    r = oracle.align_batch(a.reads_packed, a.read_off, a.read_len, a.wins_packed, a.win_off, a.win_len, a.pairs,
                           OracleScoring(), threads=2)
    # most reads are cut from their window with about 1 % substitutions: they score near their length
    assert (r.score > 480).mean() > 0.8 and (r.score < 0).sum() <= 8


@pytest.mark.gpu
def test_gpu_step3_alignment_and_choice():
    import parity
    from paper_1302_5507_b200 import Context
    sc = OracleScoring()
    b = W.make_step3(600, max_candidates=30, ref_bases=1_000_000)
    with Context(device=0) as ctx:
        parity.check_batch(ctx, b, sc, "step-3 shape", host_path=False)
        db = ctx.upload(b)
        res = ctx.align_batch(db)
        got = ctx.best_per_read(db, res)
        score = ctx.fetch(res).score
    exp = oracle.best_per_read(b.pairs, score, len(b.read_len))
    for k in exp:
        assert np.array_equal(exp[k].astype(np.int64), got[k].astype(np.int64)), k
    # the true window (or an overlapping shifted copy that still holds the read) wins almost always
    assert (got["best_score"] > 60).mean() > 0.9


@pytest.mark.gpu
def test_gpu_best_per_read_rejects_foreign_result():
    from paper_1302_5507_b200 import Context, SdpError
    b1 = W.make_step3(50, ref_bases=300_000)
    b2 = W.make_step3(60, ref_bases=300_000)
    with Context(device=0) as ctx:
        d1, d2 = ctx.upload(b1), ctx.upload(b2)
        r1 = ctx.align_batch(d1)
        ctx.align_batch(d2)
        with pytest.raises(SdpError):
            ctx.best_per_read(d1, r1)


@pytest.mark.gpu
def test_gpu_screen_then_align_winners():
    # the step-3 flow: score every candidate (forward pass only), choose per read, align only the winners
    from paper_1302_5507_b200 import Context
    sc = OracleScoring()
    b = W.make_step3(400, max_candidates=30, ref_bases=1_000_000)
    full = oracle.align_batch(b.reads_packed, b.read_off, b.read_len, b.wins_packed, b.win_off, b.win_len, b.pairs, sc,
                              threads=4)
    exp_best = oracle.best_per_read(b.pairs, full.score, len(b.read_len))
    with Context(device=0) as ctx:
        ctx.set_score_only(True)
        db = ctx.upload(b)
        res = ctx.align_batch(db)
        scr = ctx.fetch(res)
        assert np.array_equal(scr.score, full.score) and np.array_equal(scr.ref_end, full.ref_end)
        assert not scr.cigar_len.any() and not scr.passed.any() and (scr.ref_start == -1).all() and len(scr.cigar_ops) == 0
        best = ctx.best_per_read(db, res)
        for k in exp_best:
            assert np.array_equal(exp_best[k].astype(np.int64), best[k].astype(np.int64)), k
        ctx.set_score_only(False)
        winners = b.subset(best["best_pair"].astype(np.int64))
        got = ctx.fetch(ctx.align_batch(ctx.upload(winners)))
    w = best["best_pair"].astype(np.int64)
    for f in ("score", "ref_start", "ref_end", "n_match", "n_cols", "passed", "cigar_len"):
        assert np.array_equal(np.asarray(getattr(full, f))[w].astype(np.int64), getattr(got, f).astype(np.int64)), f
    for i, p in enumerate(w):
        assert full.cigar(int(p)) == got.cigar(i)
