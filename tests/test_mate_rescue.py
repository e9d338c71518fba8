"""mate-rescue wrapper (window from the mapped end and the fragment-length bounds; properly-paired flag).

CPU: pins the oracle restatement with hand-computed cases and with fragments drawn forward from the model. GPU:
sdp_mate_windows / sdp_proper_pairs against the oracle, end to end through an alignment."""
import numpy as np
import pytest

import oracle
from oracle import OracleScoring
from paper_1302_5507_b200 import workloads as W


def test_hand_computed_windows():
    # min 400, max 600, read 100: mate forward at 1000 -> [1000+400-100, 1000+600) = [1300, 1600)
    # mate reverse at [5000, 5100) -> [5100-600, 5100-400+100) = [4500, 4800); clipping at both reference ends
    off, ln = oracle.mate_windows([1000, 5000, 50, 9900, 20], [100, 100, 100, 100, 100], [0, 1, 1, 0, 1], [100] * 5, 400, 600,
                                  10_000)
    assert list(off) == [1300, 4500, 0, 0, 0] and list(ln) == [300, 300, 0, 0, 0]


def test_every_model_fragment_falls_inside_the_window():
    rng = np.random.default_rng(3)
    for _ in range(2000):
        n, L = int(rng.integers(30, 200)), int(rng.integers(30, 200))
        lo_i, hi_i = 300, 700
        ins = int(rng.integers(max(lo_i, n, L), hi_i + 1))
        f = int(rng.integers(1000, 50_000))                     # far from the reference ends: no clipping
        if rng.random() < 0.5:          # mapped end = forward end [f, f+L), other end = [f+ins-n, f+ins)
            p, rev, other = f, 0, (f + ins - n, f + ins)
        else:                           # mapped end = reverse end [f+ins-L, f+ins), other end = [f, f+n)
            p, rev, other = f + ins - L, 1, (f, f + n)
        off, ln = oracle.mate_windows([p], [L], [rev], [n], lo_i, hi_i, 10**9)
        assert off[0] <= other[0] and other[1] <= off[0] + ln[0]
        # and the implied fragment length of the true placement is ins -> properly paired
        pp = oracle.proper_pairs([p], [L], [rev], lo_i, hi_i, off, ln, [other[0] - off[0]], [other[1] - 1 - off[0]], [1])
        assert pp[0] == 1
        # the window is tight: one base outside either end would admit a fragment outside the bounds
        assert ln[0] == (hi_i - lo_i) + n


def test_hand_computed_proper_pair_rejections():
    """Negative pins of oracle.proper_pairs (reading R17), every expected value computed by hand. Bounds 400..600,
    mapped end of 100 bases, window [1300, 1600) for a forward mate at 1000, [4500, 4800) for a reverse mate at [5000, 5100)."""
    lo, hi = 400, 600
    # forward mate at p = 1000: ins = (win_off + ref_end + 1) - p
    fw = lambda ref_end, passed=1, win_len=300: int(oracle.proper_pairs([1000], [100], [0], lo, hi, [1300], [win_len], [0],
                                                                        [ref_end], [passed])[0])
    assert fw(299) == 1                  # ins = 1300 + 299 + 1 - 1000 = 600 = max: accepted
    assert fw(99) == 1                   # ins = 400 = min: accepted
    assert fw(300) == 0                  # ins = 601 = max + 1
    assert fw(98) == 0                   # ins = 399 = min - 1
    assert fw(199, passed=0) == 0        # ins = 500 but the similarity filter failed
    assert fw(199, win_len=0) == 0       # no window left after clipping: never aligned
    assert fw(199) == 1                  # the same placement with nothing wrong
    # reverse mate at [5000, 5100): ins = (p + L) - (win_off + ref_start)
    rv = lambda ref_start: int(oracle.proper_pairs([5000], [100], [1], lo, hi, [4500], [300], [ref_start], [ref_start + 99],
                                                   [1])[0])
    assert rv(0) == 1                    # ins = 5100 - 4500 = 600
    assert rv(200) == 1                  # ins = 400
    assert rv(201) == 0                  # one base too far right: ins = 399
    # one base left of the window cannot be reported (ref_start >= 0); with a window that starts earlier it is rejected
    assert int(oracle.proper_pairs([5000], [100], [1], lo, hi, [4400], [400], [99], [198], [1])[0]) == 0     # ins = 601
    assert int(oracle.proper_pairs([5000], [100], [1], lo, hi, [4400], [400], [100], [199], [1])[0]) == 1    # ins = 600


def test_mate_pairs_skip_empty_windows():
    pairs, por = oracle.mate_pairs([300, 0, 120, 0, 0, 7])
    assert pairs.tolist() == [[0, 0], [2, 2], [5, 5]]
    assert por.tolist() == [0, 0xFFFFFFFF, 1, 0xFFFFFFFF, 0xFFFFFFFF, 2]
    # results are indexed through pair_of_rescue: rescue 2 reads entry 1 of the result arrays
    pp = oracle.proper_pairs([1000, 0, 1000, 0, 0, 1000], [100] * 6, [0] * 6, 400, 600, [1300, 0, 1300, 0, 0, 1300],
                             [300, 0, 120, 0, 0, 7], [0, 0, 0], [199, 99, 98], [1, 1, 1], pair_of_rescue=por)
    assert pp.tolist() == [1, 0, 1, 0, 0, 0]


@pytest.mark.gpu
def test_gpu_mate_rescue_with_clipped_and_empty_windows():
    """Rescues near both reference ends: some windows are clipped, some empty. windows -> pairs -> align -> proper."""
    import torch
    from paper_1302_5507_b200 import Context
    rng = np.random.default_rng(21)
    ref_bases, P, n, L = 200_000, 4000, 100, 100
    ref_packed, _ = W.reference(ref_bases, W.SEED_BASE + 2, with_n=False)
    lo_i, hi_i = 350, 650
    rev = rng.integers(0, 2, P).astype(np.uint8)
    # a third of the mapped ends within 700 bases of either reference end
    where = rng.integers(0, 3, P)
    mate_pos = np.where(where == 0, rng.integers(0, 700, P),
                        np.where(where == 1, rng.integers(ref_bases - 800, ref_bases - L, P),
                                 rng.integers(0, ref_bases - L, P))).astype(np.int64)
    e_off, e_len = oracle.mate_windows(mate_pos, np.full(P, L), rev, np.full(P, n), lo_i, hi_i, ref_bases)
    assert (e_len == 0).sum() > 20 and ((e_len > 0) & (e_len < hi_i - lo_i + n)).sum() > 100
    dev = torch.device("cuda", 0)
    t = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a).astype(dt)).to(dev)
    mp, ml, mr, rl = t(mate_pos, np.int64), t(np.full(P, L), np.int32), t(rev, np.uint8), t(np.full(P, n), np.int32)
    # the unmapped end: a copy of the reference somewhere inside the window when the window can hold it, else random
    reads = []
    for k in range(P):
        if e_len[k] >= n:
            s = int(e_off[k]) + int(rng.integers(0, int(e_len[k]) - n + 1))
            reads.append(W.unpack(ref_packed, s, n))
        else:
            reads.append("".join("ACGT"[c] for c in rng.integers(0, 4, n)))
    r_packed, r_off, r_len, _ = W.pack_sequences(reads)
    with Context(device=0) as ctx:
        win_off, win_len = ctx.mate_windows(mp, ml, mr, rl, lo_i, hi_i, ref_bases)
        assert np.array_equal(win_off.cpu().numpy().astype(np.uint64), e_off)
        assert np.array_equal(win_len.cpu().numpy().astype(np.uint32), e_len)
        pairs, por = ctx.mate_pairs(win_len)
        e_pairs, e_por = oracle.mate_pairs(e_len)
        assert np.array_equal(pairs.cpu().numpy().astype(np.uint32), e_pairs)
        assert np.array_equal(por.cpu().numpy().astype(np.uint32), e_por)
        e_len_safe = e_len.copy()
        batch = W.Batch(r_packed, r_off, r_len, ref_packed, e_off, e_len_safe, e_pairs)
        res = ctx.align_batch(ctx.upload(batch))
        got = ctx.fetch(res)
        proper = ctx.proper_pairs(mp, ml, mr, rl, lo_i, hi_i, win_off, win_len, res, pair_of_rescue=por).cpu().numpy()
    exp_align = oracle.align_batch(r_packed, r_off, r_len, ref_packed, e_off, e_len_safe, e_pairs, OracleScoring(), threads=8)
    assert np.array_equal(exp_align.score, got.score) and np.array_equal(exp_align.ref_start, got.ref_start)
    exp = oracle.proper_pairs(mate_pos, np.full(P, L), rev, lo_i, hi_i, e_off, e_len, exp_align.ref_start, exp_align.ref_end,
                              exp_align.passed, pair_of_rescue=e_por)
    assert np.array_equal(proper, exp)
    assert (proper[e_len == 0] == 0).all() and proper.sum() > 0 and (proper == 0).sum() > (e_len == 0).sum()


@pytest.mark.gpu
def test_gpu_mate_rescue_flow():
    import torch
    from paper_1302_5507_b200 import Context
    rng = np.random.default_rng(8)
    ref_bases, P, n, L = 2_000_000, 3000, 100, 100
    ref_packed, _ = W.reference(ref_bases, W.SEED_BASE + 2, with_n=False)
    ins = np.clip(np.rint(rng.normal(500, 50, P)), 150, 900).astype(np.int64)
    f = rng.integers(0, ref_bases - 1000, P)
    rev = rng.integers(0, 2, P).astype(np.uint8)
    mate_pos = np.where(rev == 0, f, f + ins - L)
    true_start = np.where(rev == 0, f + ins - n, f)                   # where the unmapped end really lies
    lo_i, hi_i = 350, 650                                             # 3 sigma: a few fragments fall outside
    dev = torch.device("cuda", 0)
    t = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a).astype(dt)).to(dev)
    mp, ml, mr, rl = t(mate_pos, np.int64), t(np.full(P, L), np.int32), t(rev, np.uint8), t(np.full(P, n), np.int32)
    with Context(device=0) as ctx:
        win_off, win_len = ctx.mate_windows(mp, ml, mr, rl, lo_i, hi_i, ref_bases)
        e_off, e_len = oracle.mate_windows(mate_pos, np.full(P, L), rev, np.full(P, n), lo_i, hi_i, ref_bases)
        assert np.array_equal(win_off.cpu().numpy().astype(np.uint64), e_off)
        assert np.array_equal(win_len.cpu().numpy().astype(np.uint32), e_len)
        assert (e_len > 0).all()
        # reads: exact copies of the reference at their true positions (forward strand), 2-bit packed back to back
        reads = [W.unpack(ref_packed, int(s), n) for s in true_start]
        r_packed, r_off, r_len, _ = W.pack_sequences(reads)
        batch = W.Batch(r_packed, r_off, r_len, ref_packed, e_off, e_len,
                        np.stack([np.arange(P, dtype=np.uint32)] * 2, axis=1))
        res = ctx.align_batch(ctx.upload(batch))
        got = ctx.fetch(res)
        proper = ctx.proper_pairs(mp, ml, mr, rl, lo_i, hi_i, win_off, win_len, res).cpu().numpy()
    exp = oracle.proper_pairs(mate_pos, np.full(P, L), rev, lo_i, hi_i, e_off, e_len, got.ref_start, got.ref_end, got.passed)
    assert np.array_equal(proper, exp)
    inside = (ins >= lo_i) & (ins <= hi_i)
    # a read whose fragment length is within the bounds is found at its true place and flagged proper
    assert (got.score[inside] == n).all() and (proper[inside] == 1).all()
    # and the rejections: a fragment outside the bounds that was still found at its true place implies an out-of-bounds
    # fragment length and is flagged 0
    at_true_place = (e_off + got.ref_start.astype(np.int64)) == true_start
    assert (~inside).sum() > 0 and (proper == 0).sum() > 0
    assert (proper[~inside & at_true_place & (got.score == n)] == 0).all()
    assert ((e_off + got.ref_start.astype(np.int64))[inside] == true_start[inside]).all()
    assert inside.mean() > 0.95      # (a fragment just outside the bounds still overlaps the window and may align with an overhang)
