"""Pins of the LOCAL (soft-clipping) oracle variant, reading R18 (-m "not gpu").

oracle_align_pair_local is checked against things other than itself: brute-force enumeration of every local
alignment for n, m <= 6 with the tie rules applied to op strings; closed forms (an exact substring embedded in junk);
the textbook special cases (longest common substring; equality with the semi-global result when nothing can be
clipped); invariants (re-scoring, local >= semi-global, clip accounting) on generated workloads; hand-computed cases."""
import random
import re

import numpy as np
import pytest

import oracle
from oracle import OracleScoring
from paper_1302_5507_b200 import workloads as W

import alignment_reference as ref

DEFAULT = OracleScoring(1, -3, 5, 2, 0.6)
SCORINGS = [DEFAULT, OracleScoring(2, -1, 1, 1, 0.6), OracleScoring(1, -1, 2, 1, 0.6), OracleScoring(3, -2, 4, 3, 0.6),
            OracleScoring(1, -4, 6, 1, 0.6), OracleScoring(2, -3, 1, 1, 0.6), OracleScoring(5, -4, 1, 1, 0.6),
            OracleScoring(3, -9, 1, 1, 0.6)]      # a mismatch costs more than an insertion next to a deletion: H == D == I ties


def sc_tuple(s):
    return (s.match, s.mismatch, s.gap_open, s.gap_extend)


def _rand_seq(rng, n, alphabet):
    return "".join(rng.choice(alphabet) for _ in range(n))


def split_cigar(cigar):
    ops = re.findall(r"(\d+)([MIDS])", cigar)
    lead = int(ops[0][0]) if ops and ops[0][1] == "S" else 0
    trail = int(ops[-1][0]) if len(ops) > 1 and ops[-1][1] == "S" else 0
    core = "".join(f"{a}{b}" for a, b in ops if b != "S")
    return lead, core, trail


@pytest.mark.parametrize("si", range(len(SCORINGS)))
def test_bruteforce_small_local(si):
    sc = SCORINGS[si]
    rng = random.Random(7000 + si)
    seen_clip = seen_gap = seen_empty = seen_ties = 0
    for case in range(220):
        alphabet = rng.choice(["AC", "AC", "ACG", "ACGT", "ACGTN", "A"])
        T, R = _rand_seq(rng, rng.randint(1, 6), alphabet), _rand_seq(rng, rng.randint(1, 5), alphabet)
        c = ref.canonical_local(T, R, sc_tuple(sc))
        r = oracle.align_pair(T, R, sc, local=True)
        for k in ("score", "ref_start", "ref_end", "read_start", "read_end", "cigar", "n_match", "n_cols"):
            assert r[k] == c[k], (T, R, sc, k, r[k], c[k])
        seen_clip += int("S" in c["cigar"] and c["score"] > 0)
        seen_gap += int("I" in c["cigar"] or "D" in c["cigar"])
        seen_empty += int(c["score"] == 0)
        seen_ties += int(c.get("n_maximisers", 0) > 1)
    assert seen_clip > 20 and seen_empty > 0 and seen_ties > 20


@pytest.mark.parametrize("sc", [OracleScoring(2, -1, 1, 1, 0.6), OracleScoring(2, -3, 1, 1, 0.6), OracleScoring(5, -4, 1, 1, 0.6),
                                OracleScoring(3, -3, 1, 2, 0.6), OracleScoring(3, -9, 1, 1, 0.6)], ids=lambda s: f"{s.match}_{s.mismatch}_{s.gap_open}_{s.gap_extend}")
def test_bruteforce_small_local_with_indels(sc):
    # brute-force sized pairs that differ by one inserted or deleted base (cheap gaps): the D and I branches of the walk,
    # gap placement in repeats, and "opened here" before "extended" are all decided against the enumeration
    rng = random.Random(hash((sc.match, sc.mismatch)) & 0xFFFF)
    seen_d = seen_i = 0
    for case in range(300):
        alphabet = rng.choice(["AC", "ACG", "ACGT"])
        if rng.random() < 0.5:
            R = _rand_seq(rng, rng.randint(4, 5), alphabet)
            k = rng.randint(2, len(R) - 2)
            T = (R[:k] + _rand_seq(rng, rng.randint(1, 2), alphabet) + R[k:])[:7]    # the read lacks window bases: D
        else:
            R = _rand_seq(rng, rng.randint(5, 6), alphabet)
            k = rng.randint(2, len(R) - 3)
            T = R[:k] + R[k + 1:]                                                    # the read has an extra base: I
        c = ref.canonical_local(T, R, sc_tuple(sc))
        r = oracle.align_pair(T, R, sc, local=True)
        for key in ("score", "ref_start", "ref_end", "read_start", "read_end", "cigar", "n_match", "n_cols"):
            assert r[key] == c[key], (T, R, sc, key, r[key], c[key])
        seen_d += int("D" in c["cigar"])
        seen_i += int("I" in c["cigar"])
    assert seen_d >= 4 and seen_i >= 4, (seen_d, seen_i)


def test_hand_computed_local_cases():
    sc = DEFAULT
    # exact 7-mer inside junk on both sides of both sequences: 7 matches, clips 3 + 3
    r = oracle.align_pair("TTTTACGTACGTTTTT", "GGGACGTACGGGG", sc, local=True)
    assert (r["score"], r["ref_start"], r["ref_end"], r["read_start"], r["read_end"], r["cigar"]) == (7, 4, 10, 3, 9, "3S7M3S")
    assert (r["n_match"], r["n_cols"], r["pass"]) == (7, 7, 0)            # 7 / (7 + 6 clipped) < 0.6
    # nothing in common: empty alignment
    r = oracle.align_pair("CCCC", "GGGG", sc, local=True)
    assert (r["score"], r["ref_start"], r["ref_end"], r["read_start"], r["read_end"], r["cigar"], r["pass"]) == \
           (0, 0, -1, 0, -1, "4S", 0)
    # a mismatch in the middle is kept when both flanks outweigh it: 6 - 3 + 5 = 8 > 6
    r = oracle.align_pair("AAACGTACGGTCATTT", "CGTACGCTCATT", sc, local=True)
    assert (r["score"], r["cigar"], r["ref_start"], r["read_start"], r["n_match"]) == (8, "12M", 3, 0, 11)
    # ... and a flank that only mismatches is clipped: ACC against CGG scores nothing, TCATT is the alignment
    r = oracle.align_pair("AAACGTACGGTCATTT", "ACCTCATT", sc, local=True)
    assert (r["score"], r["cigar"], r["read_start"], r["read_end"]) == (5, "3S5M", 3, 7)
    # a 1-base deletion is bridged when the flanks pay for it: 10 + 10 - (5 + 2) = 13 > 10
    T = "GATTACAGCCTGAACTGGTCAATGC"
    r = oracle.align_pair(T, "TTACAGCCTGACTGGTCAAT", sc, local=True)
    assert (r["score"], r["cigar"], r["ref_start"], r["ref_end"]) == (13, "10M1D10M", 2, 22)
    # two equal hits: lowest end row wins (ends 5 and 9)
    r = oracle.align_pair("ACGTACGTAC", "GTAC", sc, local=True)
    assert (r["score"], r["ref_start"], r["ref_end"]) == (4, 2, 5)
    # one window row, two read positions: lowest end column wins
    r = oracle.align_pair("A", "CACA", sc, local=True)
    assert (r["score"], r["ref_end"], r["read_start"], r["read_end"], r["cigar"]) == (1, 0, 1, 1, "1S1M2S")
    # filter counts clipped bases as columns: 8 of 10 read bases aligned and equal -> 0.8
    r = oracle.align_pair("ACGTACGT", "ACGTACGTGG", OracleScoring(1, -3, 5, 2, 0.8), local=True)
    assert (r["cigar"], r["pass"]) == ("8M2S", 1)
    r = oracle.align_pair("ACGTACGT", "ACGTACGTGG", OracleScoring(1, -3, 5, 2, 0.800001), local=True)
    assert r["pass"] == 0
    # an empty alignment never passes, not even with the threshold at zero (0 * 1e6 >= 0 * 4 would hold)
    r = oracle.align_pair("CCCC", "GGGG", OracleScoring(1, -3, 5, 2, 0.0), local=True)
    assert (r["score"], r["n_cols"], r["pass"]) == (0, 0, 0)
    # N against N is a mismatch inside a local alignment too and is not counted as a match (R8): the two 6-mers around
    # it outweigh it, 6 - 3 + 6 = 9 > 6, so the column is aligned: 13 columns, 12 matches
    r = oracle.align_pair("ACGTCANTGCATC", "ACGTCANTGCATC", sc, local=True)
    assert (r["score"], r["cigar"], r["n_match"], r["n_cols"], r["pass"]) == (9, "13M", 12, 13, 1)
    # ... and a lone N-N column next to one flank only is clipped with the shorter side: ACGTCA | N | TG
    r = oracle.align_pair("ACGTCANTG", "ACGTCANTG", sc, local=True)
    assert (r["score"], r["cigar"], r["n_match"], r["n_cols"]) == (6, "6M3S", 6, 6)


def test_closed_form_exact_core_in_junk():
    # window over {A,C}, read = junk over {G,T} + a copy of a window substring + junk over {G,T}: the junk can never match,
    # so the optimum is exactly the copied core: len * match, with forced coordinates when the core occurs once
    rng = random.Random(5150)
    for sc in (DEFAULT, SCORINGS[3], SCORINGS[4]):
        for case in range(40):
            m, L = rng.randint(60, 200), rng.randint(12, 50)
            T = _rand_seq(rng, m, "AC")
            s = rng.randint(0, m - L)
            a, b = rng.randint(0, 15), rng.randint(0, 15)
            R = _rand_seq(rng, a, "GT") + T[s:s + L] + _rand_seq(rng, b, "GT")
            r = oracle.align_pair(T, R, sc, local=True)
            assert r["score"] == L * sc.match, (T, R)
            assert (r["read_start"], r["read_end"]) == (a, a + L - 1)
            assert r["cigar"] == (f"{a}S" if a else "") + f"{L}M" + (f"{b}S" if b else "")
            assert r["n_match"] == L and r["n_cols"] == L
            first = T.find(T[s:s + L])
            assert (r["ref_start"], r["ref_end"]) == (first, first + L - 1)      # lowest end row = first occurrence


def test_longest_common_substring_special_case():
    # match 1, every other move prohibitively expensive: the local score is the length of the longest common substring
    sc = OracleScoring(1, -1000, 1000, 1000, 0.0)
    rng = random.Random(404)
    for case in range(200):
        alphabet = rng.choice(["AC", "ACGT", "ACGTN"])
        T, R = _rand_seq(rng, rng.randint(1, 60), alphabet), _rand_seq(rng, rng.randint(1, 40), alphabet)
        r = oracle.align_pair(T, R, sc, local=True)
        assert r["score"] == ref.longest_common_substring(T, R), (T, R)
        assert r["n_match"] == r["n_cols"] == r["score"]


def test_local_vs_semiglobal_relations():
    # (1) local >= max(0, semi-global): the semi-global alignment is one of the local candidates.
    # (2) match > 0 = mismatch and free... not available here; instead: when the read is an exact copy, both agree.
    # (3) when mismatch = 0 and gaps are unaffordable the local score has a closed form: the largest number of equal
    #     bases on any diagonal of the two sequences, overhanging diagonals included (counted here directly).
    rng = random.Random(77)
    for case in range(150):
        T, R = _rand_seq(rng, rng.randint(5, 80), "ACGT"), _rand_seq(rng, rng.randint(1, 40), "ACGT")
        sg = oracle.align_pair(T, R, DEFAULT)
        lo = oracle.align_pair(T, R, DEFAULT, local=True)
        assert lo["score"] >= max(0, sg["score"])
    for case in range(60):
        T = _rand_seq(rng, rng.randint(30, 120), "ACGT")
        s = rng.randint(0, len(T) - 20)
        R = T[s:s + rng.randint(8, 20)]
        sg = oracle.align_pair(T, R, DEFAULT)
        lo = oracle.align_pair(T, R, DEFAULT, local=True)
        for k in ("score", "ref_start", "ref_end", "cigar", "n_match", "n_cols", "pass"):
            assert sg[k] == lo[k], (T, R, k)
        assert (lo["read_start"], lo["read_end"]) == (0, len(R) - 1)
    sc = OracleScoring(1, 0, 1000, 1000, 0.0)
    for case in range(100):
        T, R = _rand_seq(rng, rng.randint(20, 60), "ACG"), _rand_seq(rng, rng.randint(1, 20), "ACG")
        diag_best = max(sum(1 for j in range(len(R)) if 0 <= j + d < len(T) and T[j + d] == R[j])
                        for d in range(-len(R) + 1, len(T)))
        lo = oracle.align_pair(T, R, sc, local=True)
        assert lo["score"] == diag_best and lo["n_match"] == diag_best
        assert oracle.align_pair(T, R, sc)["score"] <= lo["score"]


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_local_invariants_on_configs(cfg):
    b = W.make_config(cfg, n_pairs=100, ref_bases=400_000)
    sc = DEFAULT
    res = oracle.align_batch(b.reads_packed, b.read_off, b.read_len, b.wins_packed, b.win_off, b.win_len, b.pairs, sc,
                             read_nmask=b.read_nmask, win_nmask=b.win_nmask, threads=4, local=True)
    sg = oracle.align_batch(b.reads_packed, b.read_off, b.read_len, b.wins_packed, b.win_off, b.win_len, b.pairs, sc,
                            read_nmask=b.read_nmask, win_nmask=b.win_nmask, threads=4)
    q = int(np.floor(sc.min_similarity * 1e6 + 0.5))
    n_clipped_pairs = 0
    for p in range(b.n_pairs):
        ri, wi = b.pairs[p]
        n, m = int(b.read_len[ri]), int(b.win_len[wi])
        R = W.unpack(b.reads_packed, int(b.read_off[ri]), n, b.read_nmask)
        T = W.unpack(b.wins_packed, int(b.win_off[wi]), m, b.win_nmask)
        S, cig = int(res.score[p]), res.cigar(p)
        lead, core, trail = split_cigar(cig)
        ops = ref.expand(core)
        assert 0 <= S <= n * sc.match and S >= sg.score[p]
        one = oracle.align_pair(T, R, sc, local=True)                    # batch path == single-pair path
        assert (one["score"], one["ref_start"], one["ref_end"], one["read_start"], one["read_end"], one["cigar"]) == \
               (S, res.ref_start[p], res.ref_end[p], res.read_start[p], res.read_end[p], cig)
        if S == 0:
            assert cig == f"{n}S" and res.ref_end[p] == -1 and res.passed[p] == 0
            continue
        assert lead == res.read_start[p] and trail == n - 1 - res.read_end[p]
        assert ops.count("M") + ops.count("I") == res.read_end[p] - res.read_start[p] + 1
        assert ops.count("M") + ops.count("D") == res.ref_end[p] - res.ref_start[p] + 1
        assert ops[0] == "M" and ops[-1] == "M"
        assert ref.score_ops_from(T, R, int(res.ref_start[p]), int(res.read_start[p]), ops, sc_tuple(sc)) == S
        # no prefix of the alignment scores <= 0 (the walk would have stopped there) and no suffix either (the end would be earlier)
        for k in range(1, len(ops)):
            if ops[k - 1] == "M" and ops[k] == "M":
                ni, nj = k - ops[:k].count("I"), k - ops[:k].count("D")
                assert ref.score_ops_from(T, R, int(res.ref_start[p]), int(res.read_start[p]), ops[:k], sc_tuple(sc)) > 0
                assert ref.score_ops_from(T, R, int(res.ref_start[p]) + ni, int(res.read_start[p]) + nj, ops[k:], sc_tuple(sc)) > 0
        assert res.n_cols[p] == len(ops) and res.n_match[p] <= ops.count("M")
        assert res.passed[p] == int(int(res.n_match[p]) * 10**6 >= q * (int(res.n_cols[p]) + lead + trail))
        n_clipped_pairs += int(lead + trail > 0)
    if cfg in (1, 2, 4, 5):
        assert n_clipped_pairs > 0
