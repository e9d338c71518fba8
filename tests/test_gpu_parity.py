"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI, against the CPU oracle,
element by element on the same seeded inputs. Sizes span several tiles and ragged tails."""
import random

import numpy as np
import pytest

from oracle import OracleScoring
from paper_1302_5507_b200 import Context, SdpError, workloads as W

import parity

pytestmark = pytest.mark.gpu
DEFAULT = OracleScoring(1, -3, 5, 2, 0.6)


def make_ctx(sc: OracleScoring):
    return Context(sc.match, sc.mismatch, sc.gap_open, sc.gap_extend, sc.min_similarity, device=0)


@pytest.fixture(scope="module")
def ctx():
    c = make_ctx(DEFAULT)
    yield c
    c.destroy()


def load_golden():
    import os
    rows = []
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "worked_examples.txt")):
        f = line.split()
        if f and not f[0].startswith("#") and f[0] != "E1_LAST_ROW":
            rows.append(f)
    return rows


def test_worked_examples(ctx):
    rows = load_golden()
    b = W.batch_from_strings([r[1] for r in rows], [r[2] for r in rows])
    exp, got = parity.check_batch(ctx, b, DEFAULT, "worked examples")
    for k, r in enumerate(rows):
        assert (got.score[k], got.ref_start[k], got.ref_end[k], got.cigar(k)) == (int(r[3]), int(r[4]), int(r[5]), r[6])


@pytest.mark.parametrize("cfg,n_pairs", [(1, 1000), (2, 3000), (3, 2500), (4, 1500), (5, 6000)])
def test_configs_small(ctx, cfg, n_pairs):
    # config 1 at its full size; the others shrunk so the oracle finishes in seconds
    b = W.make_config(cfg, n_pairs=n_pairs, ref_bases=2_000_000)
    parity.check_batch(ctx, b, DEFAULT, f"cfg{cfg}")


def test_ragged_counts(ctx):
    # pair counts around the warp-task sizes (16 pairs per warp at n=100, 4 warps per CTA)
    full = W.make_config(2, n_pairs=200, ref_bases=500_000)
    for cnt in (1, 2, 3, 15, 16, 17, 31, 33, 63, 64, 65, 129):
        parity.check_batch(ctx, full.subset(np.arange(cnt)), DEFAULT, f"count={cnt}", host_path=False)


@pytest.mark.parametrize("chunks", [1, 2, 3, 5, 8])
def test_chunked_lanes(chunks):
    # sdp_set_chunks: the pair list split into pipelined lanes; every output array (the CIGAR offsets run across the
    # lanes) must be what the unsplit call gives. Also a batch with fewer pairs than lanes, and mixed read lengths.
    c = make_ctx(DEFAULT)
    try:
        c.set_chunks(chunks)
        for cfg, n_pairs in ((2, 3001), (5, 4000), (4, 700), (1, 3)):
            b = W.make_config(cfg, n_pairs=n_pairs, ref_bases=1_000_000)
            parity.check_batch(c, b, DEFAULT, f"cfg{cfg} in {chunks} lanes")
        with pytest.raises(SdpError):
            c.set_chunks(9)
    finally:
        c.destroy()


def test_empty_batch(ctx):
    full = W.make_config(1, n_pairs=4, ref_bases=100_000)
    b = full.subset(np.arange(0))
    got = ctx.fetch(ctx.align_batch(ctx.upload(b)))
    assert got.score.shape == (0,) and got.cigar_ops.shape == (0,)
    got = ctx.align_batch_host(b)
    assert got.score.shape == (0,)


def test_shuffled_and_repeated_pairs(ctx):
    # many windows per read and a permuted pair list: results must follow caller order
    b = W.make_config(5, n_pairs=400, ref_bases=500_000)
    rng = np.random.default_rng(5)
    ri = rng.integers(0, 400, size=1500).astype(np.uint32)
    wi = rng.integers(0, 400, size=1500).astype(np.uint32)
    b2 = W.Batch(b.reads_packed, b.read_off, b.read_len, b.wins_packed, b.win_off, b.win_len,
                 np.stack([ri, wi], axis=1), b.read_nmask, b.win_nmask, "shuffled")
    parity.check_batch(ctx, b2, DEFAULT, "shuffled pairs")


def test_every_read_length(ctx):
    # every n in 1..330 (all column counts K, all group sizes G, ragged last columns) against
    # windows of assorted lengths, including windows shorter than the read
    rng = random.Random(11)
    reads, wins = [], []
    for n in range(1, 331):
        m = rng.choice([1, 2, 3, n, n + 1, n // 2 + 1, n + 37, 2 * n + 5, 400])
        T = "".join(rng.choice("ACGT") for _ in range(m))
        if m > n and rng.random() < 0.7:
            s = rng.randint(0, m - n)
            R = list(T[s:s + n])
            for _ in range(rng.randint(0, 3)):
                R[rng.randrange(n)] = rng.choice("ACGT")
            R = "".join(R)
            if n > 20 and rng.random() < 0.5:
                k = rng.randint(5, n - 5)
                R = (R[:k] + R[k + 2:] + "AC") if rng.random() < 0.5 else (R[:k] + "GT" + R[k:n - 2])
        else:
            R = "".join(rng.choice("ACGT") for _ in range(n))
        reads.append(R)
        wins.append(T)
    b = W.batch_from_strings(wins, reads)
    parity.check_batch(ctx, b, DEFAULT, "every read length")


def test_long_reads(ctx):
    rng = random.Random(12)
    reads, wins = [], []
    for n in (331, 400, 512, 700, 999, 1000, 1023, 1024):
        for rep in range(3):
            m = n + rng.randint(0, 600)
            T = "".join(rng.choice("ACGT") for _ in range(m))
            s = rng.randint(0, m - n)
            R = list(T[s:s + n])
            for _ in range(n // 50):
                R[rng.randrange(n)] = rng.choice("ACGT")
            k = rng.randint(50, n - 50)
            R = "".join(R)
            R = R[:k] + R[k + 3:] + "ACG" if rep else R
            reads.append(R)
            wins.append(T)
    b = W.batch_from_strings(wins, reads)
    parity.check_batch(ctx, b, DEFAULT, "long reads")


def test_band_widths(ctx):
    # gap bounds W from 0 to ~40 (narrow-band kernels up to W = 23, wide path beyond), reads up to the row limit
    # of the narrow-band kernels (n + W around 336), indels near both read ends, N on both sides, short windows
    rng = random.Random(21)
    reads, wins = [], []
    for rep in range(1800):
        n = rng.choice([30, 47, 64, 100, 101, 150, 200, 250, 299, 300, 310, 320, 330, 336])
        m = n + rng.choice([0, 3, 40, 300])
        T = [rng.choice("ACGT") for _ in range(m)]
        if rng.random() < 0.2:
            a = rng.randrange(m)
            for k in range(a, min(m, a + rng.randint(1, 12))):
                T[k] = "N"
        s = rng.randint(0, m - n)
        R = T[s:s + n]
        for _ in range(rng.randint(0, 20)):                       # each substitution widens W by 2
            R[rng.randrange(n)] = rng.choice("ACGT")
        for _ in range(rng.randint(0, 2)):
            k = rng.choice([rng.randint(0, 6), rng.randint(max(0, n - 7), n - 1), rng.randrange(n)])
            L = rng.randint(1, 12)
            if rng.random() < 0.5:
                R = R[:k] + [rng.choice("ACGT") for _ in range(L)] + R[k:]
            else:
                R = R[:k] + R[k + L:]
        R = (R + [rng.choice("ACGT") for _ in range(n)])[:n]
        R = [c if c != "N" else rng.choice("ACGTN") for c in R]
        reads.append("".join(R))
        wins.append("".join(T))
    b = W.batch_from_strings(wins, reads)
    parity.check_batch(ctx, b, DEFAULT, "band widths")


def test_extreme_shapes(ctx):
    # the longest windows the int16 range rule admits for n = 100, the longest reads, a single pair, 200,000 copies
    # of one pair, one read against many overlapping windows of one reference, reads longer than tiny windows
    rng = random.Random(99)

    def rnd(k):
        return "".join(rng.choice("ACGT") for _ in range(k))

    def mutate(seq, subs, indel):
        seq = list(seq)
        for _ in range(subs):
            seq[rng.randrange(len(seq))] = rng.choice("ACGT")
        if indel:
            k = rng.randrange(5, len(seq) - 5)
            seq = seq[:k] + (list(rnd(indel)) if rng.random() < 0.5 else []) + seq[k + (0 if rng.random() < 0.5 else indel):]
        return "".join(seq)

    wins, reads = [], []
    for m in (7800, 12000, 15800):
        for _ in range(4):
            T = rnd(m)
            s = rng.randrange(0, m - 100)
            reads.append(mutate(T[s:s + 100], rng.randint(0, 6), rng.choice([0, 0, 2, 7]))[:100].ljust(100, "A"))
            wins.append(T)
    parity.check_batch(ctx, W.batch_from_strings(wins, reads), DEFAULT, "longest windows")
    wins, reads = [], []
    for n in (1000, 1024):
        for _ in range(5):
            m = n + rng.randint(0, 900)
            T = rnd(m)
            s = rng.randrange(0, m - n + 1)
            reads.append((mutate(T[s:s + n], rng.randint(0, 40), rng.choice([0, 3, 15])) + rnd(n))[:n])
            wins.append(T)
    parity.check_batch(ctx, W.batch_from_strings(wins, reads), DEFAULT, "longest reads")
    T = rnd(400)
    R = mutate(T[120:220], 3, 2)[:100].ljust(100, "C")
    parity.check_batch(ctx, W.batch_from_strings([T], [R]), DEFAULT, "one pair")
    b = W.batch_from_strings([T], [R], pairs=np.zeros((200000, 2), dtype=np.uint32))
    parity.check_batch(ctx, b, DEFAULT, "200k identical pairs", host_path=False)
    ref = rnd(2000)
    R = mutate(ref[900:1050], 4, 3)[:150].ljust(150, "G")
    wins = [ref[k:k + 600] for k in range(500, 1000, 7)]
    b = W.batch_from_strings(wins, [R], pairs=np.array([[0, k] for k in range(len(wins))], dtype=np.uint32))
    parity.check_batch(ctx, b, DEFAULT, "one read, many overlapping windows")
    wins = [rnd(rng.randint(1, 20)) for _ in range(300)]
    reads = [rnd(rng.randint(1, 60)) for _ in range(300)]
    parity.check_batch(ctx, W.batch_from_strings(wins, reads), DEFAULT, "reads longer than tiny windows")


def test_n_bases_both_sides(ctx):
    rng = random.Random(13)
    reads, wins = [], []
    for _ in range(300):
        n, m = rng.randint(20, 120), rng.randint(60, 300)
        T = [rng.choice("ACGT") for _ in range(m)]
        for _ in range(rng.randint(0, 3)):
            a = rng.randrange(m)
            for k in range(a, min(m, a + rng.randint(1, 30))):
                T[k] = "N"
        s = rng.randint(0, max(0, m - n))
        R = (T[s:s + n] + [rng.choice("ACGT") for _ in range(n)])[:n]
        R = [c if c != "N" or rng.random() < 0.5 else rng.choice("ACGT") for c in R]
        for _ in range(rng.randint(0, 2)):
            R[rng.randrange(n)] = "N"
        reads.append("".join(R))
        wins.append("".join(T))
    wins.append("N" * 40)
    reads.append("ACGTACGTAC")          # all-N window: all-insertion alignment, span 0
    b = W.batch_from_strings(wins, reads)
    assert b.read_nmask is not None and b.win_nmask is not None
    parity.check_batch(ctx, b, DEFAULT, "N bases")


def test_tie_heavy_low_complexity(ctx):
    rng = random.Random(14)
    reads, wins = [], []
    for _ in range(600):
        alpha = rng.choice(["A", "AC", "AC", "ACG"])
        n, m = rng.randint(1, 40), rng.randint(1, 90)
        wins.append("".join(rng.choice(alpha) for _ in range(m)))
        reads.append("".join(rng.choice(alpha) for _ in range(n)))
    b = W.batch_from_strings(wins, reads)
    parity.check_batch(ctx, b, DEFAULT, "low complexity")


@pytest.mark.parametrize("sc", [OracleScoring(2, -1, 1, 1, 0.5), OracleScoring(1, -1, 2, 1, 0.7),
                                OracleScoring(3, -2, 4, 3, 0.6), OracleScoring(1, -4, 6, 1, 0.9),
                                OracleScoring(1, -9, 1, 1, 0.6), OracleScoring(0, -1, 0, 1, 0.0),
                                OracleScoring(5, -4, 0, 1, 0.6), OracleScoring(1, 0, 3, 2, 0.6)],
                         ids=lambda s: f"{s.match}_{s.mismatch}_{s.gap_open}_{s.gap_extend}")
def test_other_scorings(sc):
    c = make_ctx(sc)
    try:
        b = W.make_config(4, n_pairs=300, ref_bases=300_000)
        parity.check_batch(c, b, sc, f"scoring {sc}", host_path=False)
        rng = random.Random(15)
        wins = ["".join(rng.choice("AC") for _ in range(rng.randint(1, 60))) for _ in range(300)]
        reads = ["".join(rng.choice("AC") for _ in range(rng.randint(1, 30))) for _ in range(300)]
        parity.check_batch(c, W.batch_from_strings(wins, reads), sc, f"scoring {sc} ties", host_path=False)
    finally:
        c.destroy()


@pytest.mark.parametrize("sc", [OracleScoring(20, -60, 100, 40, 0.6), OracleScoring(1, -3, 5, 400, 0.6),
                                OracleScoring(1, -3, 2000, 2, 0.6), OracleScoring(1, -4000, 5, 2, 0.6),
                                OracleScoring(250, -3, 5, 375, 0.6), OracleScoring(4000, -4000, 4000, 4000, 0.6),
                                OracleScoring(200, -39, 3, 1, 0.6), OracleScoring(240, 0, 7, 3, 0.6)],
                         ids=lambda s: f"{s.match}_{s.mismatch}_{s.gap_open}_{s.gap_extend}")
def test_scorings_at_the_accepted_extremes(sc):
    # large constants: the int16 range rule, the fp16 bit-pattern tricks (match - mismatch up to 8000, 8 times
    # that in the tagged traceback kernels) and the patched immediates near their limits; pairs that leave the int16
    # domain must take the int32 lane and the generic band kernel, never a wrong fast path
    c = make_ctx(sc)
    try:
        for cfg, n_pairs in ((2, 400), (4, 200), (5, 400)):
            parity.check_batch(c, W.make_config(cfg, n_pairs=n_pairs, ref_bases=300_000), sc, f"cfg{cfg} scoring {sc}",
                               host_path=False)
        rng = random.Random(16)
        wins = ["".join(rng.choice("ACGT") for _ in range(rng.randint(1, 80))) for _ in range(200)]
        reads = ["".join(rng.choice("ACGT") for _ in range(rng.randint(1, 40))) for _ in range(200)]
        parity.check_batch(c, W.batch_from_strings(wins, reads), sc, f"scoring {sc} short", host_path=False)
    finally:
        c.destroy()


@pytest.mark.parametrize("route", [dict(no_thin=True), dict(no_wide=True), dict(no_thin=True, no_wide=True),
                                   dict(always_reverse=True), dict(no_thin=True, always_reverse=True)],
                         ids=["no_thin", "no_wide", "generic_only", "always_reverse", "no_thin_always_reverse"])
def test_alternative_traceback_paths(route):
    # route the same pairs through the other traceback kernels (wide wavefront for every W >= 1; generic scalar band
    # kernel instead of the wavefront; generic kernel for everything; the reverse pass for every wide pair instead of
    # only where it pays): all must agree with the oracle
    c = make_ctx(DEFAULT)
    try:
        c.set_debug_route(**route)
        parity.check_batch(c, W.make_config(3, n_pairs=1200, ref_bases=500_000), DEFAULT, f"cfg3 {route}", host_path=False)
        parity.check_batch(c, W.make_config(5, n_pairs=1500, ref_bases=500_000), DEFAULT, f"cfg5 {route}", host_path=False)
        parity.check_batch(c, W.make_config(4, n_pairs=600, ref_bases=500_000), DEFAULT, f"cfg4 {route}", host_path=False)
        parity.check_batch(c, W.make_config(2, n_pairs=2000, ref_bases=500_000), DEFAULT, f"cfg2 {route}", host_path=False)
        c.set_debug_route()                                   # back to the default routing
        parity.check_batch(c, W.make_config(5, n_pairs=700, ref_bases=500_000), DEFAULT, "cfg5 default route", host_path=False)
    finally:
        c.destroy()


@pytest.mark.parametrize("g", [1, 2, 3, 5, 8, 16, 32])
def test_forced_group_sizes(g):
    # every thread-group size G the geometry table can pick, forced for all read lengths that admit it
    c = make_ctx(DEFAULT)
    try:
        c.set_debug_route(force_g=g)
        parity.check_batch(c, W.make_config(5, n_pairs=2500, ref_bases=500_000), DEFAULT, f"cfg5 G={g}", host_path=False)
        parity.check_batch(c, W.make_config(1, n_pairs=300, ref_bases=200_000), DEFAULT, f"cfg1 G={g}", host_path=False)
    finally:
        c.destroy()


@pytest.mark.parametrize("sc", [DEFAULT, OracleScoring(2, -1, 1, 1, 0.5), OracleScoring(1, -4, 6, 1, 0.9), OracleScoring(1, -1, 9, 3, 0.6)],
                         ids=lambda s: f"{s.match}_{s.mismatch}_{s.gap_open}_{s.gap_extend}")
def test_prefilter_changes_nothing(sc):
    # the ungapped pre-pass (sdp_set_prefilter) settles near-exact pairs without DP; every output must stay bit-exact.
    # Scorings: at most 1 / 0 / 1 / 5 mismatches allowed by x*(match-mismatch) < open+extend
    c = make_ctx(sc)
    try:
        c.set_prefilter(True)
        for cfg, P in ((2, 3000), (5, 4000), (3, 1500)):
            parity.check_batch(c, W.make_config(cfg, n_pairs=P, ref_bases=500_000), sc, f"prefilter cfg{cfg}")
            st = c.stats()
            assert st["cells_prefiltered"] > 0 or sc.mismatch == -1 and sc.match == 2
        rng = random.Random(31)
        wins = ["".join(rng.choice("AC") for _ in range(rng.randint(1, 80))) for _ in range(500)]     # ties everywhere
        reads = ["".join(rng.choice("AC") for _ in range(rng.randint(1, 30))) for _ in range(500)]
        parity.check_batch(c, W.batch_from_strings(wins, reads), sc, "prefilter low complexity", host_path=False)
        wins = ["ACGTNNACGTACGTNACGTACGTAAC" * 3 for _ in range(40)]
        reads = [w[k:k + 20] for k, w in enumerate(wins)]
        parity.check_batch(c, W.batch_from_strings(wins, reads), sc, "prefilter with N", host_path=False)
    finally:
        c.destroy()


def test_mixed_window_lengths_in_one_warp(ctx):
    # same read length, window lengths from 1 to 900 in one batch: lanes of a warp finish at
    # different rows (the masked tail loop of the score kernel)
    rng = random.Random(16)
    T0 = "".join(rng.choice("ACGT") for _ in range(2000))
    reads, wins = [], []
    for k in range(400):
        m = rng.choice([1, 5, 50, 99, 100, 101, 130, 250, 500, 899, 900])
        s = rng.randint(0, 2000 - m)
        wins.append(T0[s:s + m])
        a = rng.randint(0, 1900)
        reads.append(T0[a:a + 100])
    parity.check_batch(ctx, W.batch_from_strings(wins, reads), DEFAULT, "mixed m")


@pytest.mark.parametrize("cfg,n_pairs", [(1, 1000), (2, 2500), (3, 1500), (4, 800), (5, 3000)])
def test_local_mode_configs(cfg, n_pairs):
    # the soft-clipping variant on all five configs; read_start / read_end are no longer constants
    c = make_ctx(DEFAULT)
    try:
        c.set_mode(local=True)
        b = W.make_config(cfg, n_pairs=n_pairs, ref_bases=2_000_000)
        exp, got = parity.check_batch(c, b, DEFAULT, f"local cfg{cfg}", local=True)
        n = b.read_len[b.pairs[:, 0]].astype(np.int64)
        clipped = (got.read_start > 0) | (got.read_end < n - 1)
        assert clipped.any() and (~clipped).any()
        assert ((got.cigar_ops & 15) == 4).any()
        c.set_mode(local=False)                                  # and back: the semi-global results are unchanged
        parity.check_batch(c, b.subset(np.arange(min(300, b.n_pairs))), DEFAULT, f"semi-global after local cfg{cfg}",
                           host_path=False)
    finally:
        c.destroy()


def test_local_mode_edges():
    rng = random.Random(61)
    wins, reads = [], []
    for _ in range(500):                                         # ties, empty alignments, N, tiny sizes
        alpha = rng.choice(["A", "AC", "AC", "ACG", "ACGTN"])
        wins.append("".join(rng.choice(alpha) for _ in range(rng.randint(1, 70))))
        reads.append("".join(rng.choice(alpha) for _ in range(rng.randint(1, 40))))
    wins += ["CCCC", "A", "ACGTACGTAC", "TTTTACGTACGTTTTT", "ACGTCANTGCATC", "ACGTCANTG"]
    reads += ["GGGG", "CACA", "GTAC", "GGGACGTACGGGG", "ACGTCANTGCATC", "ACGTCANTG"]     # N against N inside / beside an alignment
    for sc in (DEFAULT, OracleScoring(2, -1, 1, 1, 0.5), OracleScoring(3, -9, 1, 1, 0.6), OracleScoring(1, -4, 6, 1, 0.9),
               OracleScoring(1, -3, 5, 2, 0.0)):                      # threshold 0: an empty alignment still fails the filter
        c = make_ctx(sc)
        try:
            c.set_mode(local=True)
            exp, got = parity.check_batch(c, W.batch_from_strings(wins, reads), sc, f"local edges {sc}", local=True)
            assert (got.score == 0).any() and (got.ref_end[got.score == 0] == -1).all()
        finally:
            c.destroy()


def test_int32_lane(ctx):
    # pairs outside the int16 kernels' domain are aligned on the int32 lane instead of being rejected:
    # a 9,000-base and a 17,000-base window for a 100-base read, reads of 1,025 and 2,000 bases, mixed with ordinary pairs
    rng = random.Random(62)

    def rnd(k):
        return "".join(rng.choice("ACGT") for _ in range(k))

    def mutate(seq, subs, indel):
        seq = list(seq)
        for _ in range(subs):
            seq[rng.randrange(len(seq))] = rng.choice("ACGT")
        if indel:
            k = rng.randrange(5, len(seq) - 5)
            seq = seq[:k] + (list(rnd(indel)) if rng.random() < 0.5 else []) + seq[k + (0 if rng.random() < 0.5 else indel):]
        return "".join(seq)

    wins, reads = [], []
    for m, n in ((9000, 100), (17000, 100), (20000, 250), (3000, 1025), (2500, 2000), (1500, 1200), (600, 100), (500, 100)):
        for _ in range(3):
            T = rnd(m)
            s = rng.randrange(0, m - n + 1)
            reads.append((mutate(T[s:s + n], rng.randint(0, n // 20), rng.choice([0, 0, 3, 12])) + rnd(n))[:n])
            wins.append(T)
    reads.append(rnd(1500)); wins.append(rnd(1800))              # an unplaceable long read: widest band
    exp, got = parity.check_batch(ctx, W.batch_from_strings(wins, reads), DEFAULT, "int32 lane")
    assert ctx.stats()["n_slow_words"] > 0
    # a scoring whose constants alone leave the int16 domain for ordinary lengths
    sc = OracleScoring(300, -400, 600, 200, 0.6)
    c = make_ctx(sc)
    try:
        parity.check_batch(c, W.make_config(1, n_pairs=200, ref_bases=200_000), sc, "int32 lane, large scoring", host_path=False)
        assert c.stats()["n_slow_words"] > 0
    finally:
        c.destroy()


@pytest.mark.parametrize("route", ["local", "long_window", "large_scoring"])
def test_int32_lane_reads_257_to_1024(route):
    # reads of 257..1,024 bases on the int32 lane (forward_i32_warp<16> for 257..512, <32> for
    # 513..1,024; row arrays of up to 1,025 cells in k_traceback<1032, .>), reached in each of the three ways a pair
    # gets there: local mode, a window long enough to break the int16 range rule (PAPER.md:117,
    # sdp.h), and a scoring whose constants alone break it. Placed, gapped, clipped and unplaceable reads.
    rng = random.Random(63)

    def rnd(k):
        return "".join(rng.choice("ACGT") for _ in range(k))

    wins, reads = [], []
    for n in (257, 300, 400, 512, 513, 700, 1000, 1024):
        for kind in ("placed", "indels", "clipped", "unplaceable"):
            for _ in range(1 if route == "long_window" else 2):
                m = 16500 + rng.randint(0, 300) if route == "long_window" else n + rng.randint(40, 600)
                T = rnd(m)
                s = rng.randrange(0, m - n + 1)
                R = list(T[s:s + n])
                for _ in range(rng.randint(0, n // 25)):
                    R[rng.randrange(n)] = rng.choice("ACGT")
                if kind == "indels":
                    for _ in range(rng.randint(1, 4)):
                        k, g = rng.randrange(10, len(R) - 40), rng.randint(1, 30)
                        R = R[:k] + (list(rnd(g)) if rng.random() < 0.5 else []) + R[k + (0 if rng.random() < 0.5 else g):]
                elif kind == "clipped":                          # foreign ends: soft clips in local mode, wide bands otherwise
                    a, z = rng.randint(5, n // 3), rng.randint(5, n // 3)
                    R = list(rnd(a)) + R[a:n - z] + list(rnd(z))
                elif kind == "unplaceable":
                    R = list(rnd(n))
                reads.append(("".join(R) + rnd(n))[:n])
                wins.append(T)
    sc = OracleScoring(300, -400, 600, 200, 0.6) if route == "large_scoring" else DEFAULT
    c = make_ctx(sc)
    try:
        c.set_mode(local=route == "local")
        b = W.batch_from_strings(wins, reads)
        exp, got = parity.check_batch(c, b, sc, f"int32 lane, n = 257..1024, {route}", local=route == "local")
        assert c.stats()["n_slow_words"] == b.n_pairs           # every pair took the lane; none needs global row arrays
        if route == "local":
            n = b.read_len[b.pairs[:, 0]].astype(np.int64)
            assert ((got.read_start > 0) | (got.read_end < n - 1)).any()
    finally:
        c.destroy()


@pytest.mark.parametrize("sc", [DEFAULT, OracleScoring(2, 0, 3, 1, 0.5), OracleScoring(60, -60, 100, 40, 0.6),
                                OracleScoring(1, -1, 0, 1, 0.6), OracleScoring(120, -7, 30, 9, 0.6)],
                         ids=lambda s: f"{s.match}_{s.mismatch}_{s.gap_open}_{s.gap_extend}")
def test_local_mode_int16_pairing(sc):
    # The int16x2 local kernel (slow_lane.cu) scores pairs 2w and 2w+1 in one warp when both reads have at most 256
    # bases and the value rule holds for the larger of their lengths; everything else stays on the int32 kernels. Mixed
    # neighbours: every read length class next to every other, windows from 1 base to lengths that break the rule for
    # the larger scorings, an odd pair count, mismatch = 0 (a padded cell can then tie with a real one: it must lose).
    rng = random.Random(65)

    def rnd(k, alpha="ACGT"):
        return "".join(rng.choice(alpha) for _ in range(k))

    wins, reads = [], []
    for _ in range(301):
        n = rng.choice([1, 2, 7, 31, 64, 100, 127, 128, 129, 200, 255, 256, 257, 300, 520])
        m = rng.choice([1, 3, 40, 150, 300, 301, 640, 900, 2500])
        alpha = rng.choice(["ACGT", "ACGT", "AC", "ACGTN"])
        T = rnd(m, alpha)
        if rng.random() < 0.7 and m > 4:                         # a read that shares a stretch with its window
            a = rng.randrange(0, m - 1)
            core = T[a:a + n]
            R = (rnd(rng.randint(0, 6), alpha) + core + rnd(n, alpha))[:n]
        else:
            R = rnd(n, alpha)
        wins.append(T); reads.append(R)
    c = make_ctx(sc)
    try:
        c.set_mode(local=True)
        parity.check_batch(c, W.batch_from_strings(wins, reads), sc, f"local int16 pairing {sc}", local=True)
        # four pairs per warp (two 16-lane groups) when a whole quad has reads of at most 128 bases: every tail size
        short = [k for k in range(len(reads)) if len(reads[k]) <= 128]
        for count in (1, 2, 3, 4, 5, 6, 7, 41):
            pick = short[:count]
            parity.check_batch(c, W.batch_from_strings([wins[k] for k in pick], [reads[k] for k in pick]), sc,
                               f"local int16 quads, {count} pairs {sc}", host_path=False, local=True)
    finally:
        c.destroy()


def test_int32_range_rule():
    # beyond match*n + gap_extend*(n+2) + 2*gap_open + |mismatch| < 2^28 the int32 lane's minus infinity
    # would no longer sit below every real cell value: such a pair is SDP_ERANGE (sdp.h), and a pair just inside the
    # rule, at the largest scoring constants sdp_create accepts, is still exact.
    rng = random.Random(64)

    def rnd(k):
        return "".join(rng.choice("ACGT") for _ in range(k))

    sc = OracleScoring(4000, -4000, 4000, 4000, 0.6)
    c = make_ctx(sc)
    try:
        T = rnd(4200)
        placed = T[100:1600] + rnd(7) + T[1600:4100]             # 4,007 bases with one insertion
        b = W.batch_from_strings([rnd(40), rnd(300), T], [rnd(30000), rnd(33000), placed])
        parity.check_batch(c, b, sc, "inside the int32 range rule", host_path=False)
        assert c.stats()["n_slow_words"] > 0
        too_long = W.batch_from_strings([rnd(50), rnd(60)], [rnd(100), rnd(34000)])
        with pytest.raises(SdpError) as e:
            c.align_batch(c.upload(too_long))
        assert e.value.code == -2
        parity.check_batch(c, W.batch_from_strings([rnd(50)], [rnd(100)]), sc, "after SDP_ERANGE", host_path=False)
    finally:
        c.destroy()


def test_errors(ctx):
    b = W.make_config(1, n_pairs=10, ref_bases=100_000)
    bad = W.Batch(b.reads_packed, b.read_off, b.read_len, b.wins_packed, b.win_off, b.win_len,
                  np.array([[0, 99]], dtype=np.uint32), None, None)
    with pytest.raises(SdpError) as e:
        ctx.align_batch(ctx.upload(bad))
    assert e.value.code == -1
    # a sequence longer than SDP_MAX_SEQ_LEN is beyond even the int32 lane (lengths only: the bases are never read)
    huge = W.Batch(b.reads_packed, b.read_off, b.read_len, b.wins_packed, np.array([0], dtype=np.uint64),
                   np.array([1_000_001], dtype=np.uint32), np.array([[0, 0]], dtype=np.uint32), None, None)
    db = ctx.upload(huge)
    db.c.wins_bases = 2_000_000                                  # (pretend the buffer is that long; the call fails before reading it)
    with pytest.raises(SdpError) as e:
        ctx.align_batch(db)
    assert e.value.code == -2
    with pytest.raises(SdpError):
        ctx._check(ctx._lib.sdp_set_mode(ctx._h, 7))             # unknown mode
    with pytest.raises(SdpError):
        Context(match=1, mismatch=1)
    with pytest.raises(SdpError):
        Context(gap_extend=0)
    # the context survives errors
    parity.check_batch(ctx, b, DEFAULT, "after errors", host_path=False)


def test_stats_and_timing(ctx):
    b = W.make_config(2, n_pairs=500, ref_bases=500_000)
    ctx.set_timing(True)
    ctx.align_batch(ctx.upload(b))
    s = ctx.stats()
    ctx.set_timing(False)
    assert s["n_pairs"] == 500 and s["cells_forward"] == b.cells
    assert s["kernel_launches"] >= 8 and s["forward_launches"] >= 1
    assert s["ms_total"] > 0 and s["ms_forward"] > 0
