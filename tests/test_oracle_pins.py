"""Pins for the CPU oracle (-m "not gpu"): everything here checks oracle/ against something other
than itself -- brute-force enumeration, closed forms, CIGAR re-scoring, a textbook edit-distance
DP, and the worked examples in tests/golden/. See DESIGN.md "Oracle pins".
"""
import os
import random

import numpy as np
import pytest

import oracle
from oracle import OracleScoring
from paper_1302_5507_b200 import workloads as W

import alignment_reference as ref

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "worked_examples.txt")
DEFAULT = OracleScoring(1, -3, 5, 2, 0.6)
SCORINGS = [
    OracleScoring(1, -3, 5, 2, 0.6),     # BASELINE.json configs
    OracleScoring(2, -1, 1, 1, 0.6),     # cheap gaps: many co-optimal paths
    OracleScoring(1, -1, 2, 1, 0.6),
    OracleScoring(3, -2, 4, 3, 0.6),
    OracleScoring(1, -4, 6, 1, 0.6),     # BWA-like
    OracleScoring(1, -9, 1, 1, 0.6),     # a mismatch costs more than I+D: forces H==D==I ties
    OracleScoring(2, -3, 1, 1, 0.6),     # open-vs-extend ties inside gaps
]


def sc_tuple(s: OracleScoring):
    return (s.match, s.mismatch, s.gap_open, s.gap_extend)


def load_golden():
    rows, last_row = [], None
    for line in open(GOLDEN):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        f = line.split()
        if f[0] == "E1_LAST_ROW":
            last_row = [int(x) for x in f[1:]]
        else:
            rows.append(dict(name=f[0], T=f[1], R=f[2], score=int(f[3]), ref_start=int(f[4]),
                             ref_end=int(f[5]), cigar=f[6], n_match=int(f[7]), n_cols=int(f[8])))
    return rows, last_row


# ---------------------------------------------------------------- P8 worked examples
@pytest.mark.parametrize("row", load_golden()[0], ids=lambda r: r["name"])
def test_worked_examples(row):
    r = oracle.align_pair(row["T"], row["R"], DEFAULT)
    for k in ("score", "ref_start", "ref_end", "cigar", "n_match", "n_cols"):
        assert r[k] == row[k], (row["name"], k, r[k], row[k])
    # the stored CIGAR re-scores to the stored score, independently of the oracle
    assert ref.rescore(row["T"], row["R"], row["ref_start"], row["cigar"], sc_tuple(DEFAULT)) == row["score"]
    # and, where brute force is affordable, brute force agrees with the stored row
    if len(row["R"]) <= 6 and len(row["T"]) <= 10:
        c = ref.canonical(row["T"], row["R"], sc_tuple(DEFAULT))
        for k in ("score", "ref_start", "ref_end", "cigar", "n_match", "n_cols"):
            assert c[k] == row[k], (row["name"], "bruteforce", k, c[k], row[k])


def test_e1_last_row():
    rows, last = load_golden()
    r = oracle.align_pair("ACGTACGTAC", "GTAC", DEFAULT, want_last_row=True)
    assert list(r["last_row"]) == last
    # row 0 of the last column is the paper's base case M(0,n) = S_GO + (n-1) S_GE
    assert last[0] == -(5 + 2 * 4)


# ---------------------------------------------------------------- P1 brute force
def _rand_seq(rng, n, alphabet):
    return "".join(rng.choice(alphabet) for _ in range(n))


@pytest.mark.parametrize("si", range(len(SCORINGS)))
def test_bruteforce_small(si):
    sc = SCORINGS[si]
    rng = random.Random(1000 + si)
    n_cases = 260
    for case in range(n_cases):
        alphabet = rng.choice(["AC", "AC", "ACG", "ACGT", "ACGTN", "A"])
        n = rng.randint(1, 5)
        m = rng.randint(1, 7)
        T, R = _rand_seq(rng, m, alphabet), _rand_seq(rng, n, alphabet)
        c = ref.canonical(T, R, sc_tuple(sc))
        r = oracle.align_pair(T, R, sc)
        ctx = (T, R, sc, c, r)
        assert r["score"] == c["score"], ctx
        assert r["ref_end"] == c["ref_end"], ctx
        assert r["ref_start"] == c["ref_start"], ctx
        assert r["cigar"] == c["cigar"], ctx
        assert r["n_match"] == c["n_match"] and r["n_cols"] == c["n_cols"], ctx
        assert (r["ref_start"], ref.expand(r["cigar"])) in c["cands"], ctx


@pytest.mark.parametrize("T,R", [("CAACCAC", "CCACAC"), ("CCAAACCA", "CACACA"), ("ACAACCCAA", "CCACCA"),
                                 ("ACCCAACC", "ACACACC")])
def test_bruteforce_gap_open_vs_extend_ties(T, R):
    # inputs where "run opened here" and "run extended" tie inside a deletion (reading R6): brute
    # force must pick the shorter run, e.g. 3M1D3M rather than 1I2M2D3M
    sc = OracleScoring(2, -3, 1, 1, 0.6)
    c = ref.canonical(T, R, sc_tuple(sc))
    r = oracle.align_pair(T, R, sc)
    assert len(c["cands"]) > 1
    for k in ("score", "ref_start", "ref_end", "cigar", "n_match", "n_cols"):
        assert r[k] == c[k], (T, R, k, r[k], c[k])


def test_bruteforce_zero_open_score_only():
    # gap_open = 0: run splitting is free so op strings are ambiguous; pin score, end and validity
    sc = OracleScoring(1, -1, 0, 1, 0.6)
    rng = random.Random(77)
    for case in range(120):
        T, R = _rand_seq(rng, rng.randint(1, 6), "ACG"), _rand_seq(rng, rng.randint(1, 5), "ACG")
        c = ref.canonical(T, R, sc_tuple(sc))
        r = oracle.align_pair(T, R, sc)
        assert r["score"] == c["score"] and r["ref_end"] == c["ref_end"], (T, R, c, r)
        assert ref.rescore(T, R, r["ref_start"], r["cigar"], sc_tuple(sc)) == r["score"]


# ---------------------------------------------------------------- P2 closed forms
def _random_window(rng, m):
    return _rand_seq(rng, m, "ACGT")


@pytest.mark.parametrize("sc", [SCORINGS[0], SCORINGS[3], SCORINGS[4]], ids=["default", "3/-2/4/3", "1/-4/6/1"])
def test_closed_forms(sc):
    rng = random.Random(4242)
    o, e = sc.gap_open, sc.gap_extend
    for case in range(60):
        m, n = rng.randint(120, 300), rng.randint(40, 100)
        T = _random_window(rng, m)
        s = rng.randint(0, m - n - 12)
        exact = T[s:s + n]
        # exact copy: n * match, coordinates and CIGAR are forced
        r = oracle.align_pair(T, exact, sc)
        assert r["score"] == n * sc.match and r["cigar"] == f"{n}M"
        assert r["n_match"] == n and r["n_cols"] == n
        if T.count(exact) == 1:
            assert (r["ref_start"], r["ref_end"]) == (s, s + n - 1)
        # one central substitution: (n-1) match + mismatch
        k = rng.randint(15, n - 16)
        sub = exact[:k] + rng.choice([c for c in "ACGT" if c != exact[k]]) + exact[k + 1:]
        r = oracle.align_pair(T, sub, sc)
        assert r["score"] == (n - 1) * sc.match + sc.mismatch, (T, sub)
        assert r["cigar"] == f"{n}M" and r["n_match"] == n - 1
        # one central k-base deletion from the read: n match - (o + k e)
        gl = rng.randint(1, 3)
        pos = rng.randint(15, n - 16)
        dele = T[s:s + pos] + T[s + pos + gl:s + n + gl]
        r = oracle.align_pair(T, dele, sc)
        assert r["score"] >= n * sc.match - (o + gl * e)
        if n * sc.match - (o + gl * e) > (n - 15) * sc.match:   # the gapped alignment must win
            assert r["score"] == n * sc.match - (o + gl * e), (T, dele, r)
            assert r["n_cols"] == n + gl and r["n_match"] == n
            assert r["ref_end"] - r["ref_start"] + 1 == n + gl
        # one central k-base insertion into the read: (n-k) match - (o + k e)
        ins = exact[:pos] + _rand_seq(rng, gl, "ACGT") + exact[pos:n - gl]
        r = oracle.align_pair(T, ins, sc)
        assert r["score"] >= (n - gl) * sc.match - (o + gl * e)


# ---------------------------------------------------------------- P3 invariants on generated workloads
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_invariants_on_configs(cfg):
    b = W.make_config(cfg, n_pairs=120, ref_bases=400_000)
    sc = DEFAULT
    res = oracle.align_batch(b.reads_packed, b.read_off, b.read_len, b.wins_packed, b.win_off, b.win_len,
                             b.pairs, sc, win_nmask=b.win_nmask, threads=4)
    o, e = sc.gap_open, sc.gap_extend
    q = int(np.floor(sc.min_similarity * 1e6 + 0.5))
    for p in range(b.n_pairs):
        ri, wi = b.pairs[p]
        n, m = int(b.read_len[ri]), int(b.win_len[wi])
        R = W.unpack(b.reads_packed, int(b.read_off[ri]), n)
        T = W.unpack(b.wins_packed, int(b.win_off[wi]), m, b.win_nmask)
        cig = res.cigar(p)
        ops = ref.expand(cig)
        S = int(res.score[p])
        assert -(o + e * n) <= S <= n * sc.match
        assert ops.count("M") + ops.count("I") == n
        assert ops.count("M") + ops.count("D") == res.ref_end[p] - res.ref_start[p] + 1
        assert 0 <= res.ref_end[p] < m and 0 <= res.ref_start[p] <= res.ref_end[p] + 1
        assert res.read_start[p] == 0 and res.read_end[p] == n - 1
        assert ref.rescore(T, R, int(res.ref_start[p]), cig, sc_tuple(sc)) == S
        assert not ops.startswith("D") and not ops.endswith("D")
        runs = [c for c in cig if c in "MID"]
        assert all(a != b_ for a, b_ in zip(runs, runs[1:]))
        assert res.n_cols[p] == len(ops) and res.n_match[p] <= ops.count("M")
        assert res.passed[p] == int(int(res.n_match[p]) * 10**6 >= q * int(res.n_cols[p]))
        # batch path == single-pair path
        one = oracle.align_pair(T, R, sc)
        assert (one["score"], one["ref_start"], one["ref_end"], one["cigar"]) == \
               (S, res.ref_start[p], res.ref_end[p], cig)
        # gap-content bound used by the banded traceback: ins+del <= W
        Wb = max(0, (n * sc.match - S - o) // e) if n * sc.match - S - o >= 0 else 0
        assert ops.count("I") + ops.count("D") <= Wb


# ---------------------------------------------------------------- P4 / P5 reverse and restriction
def test_reverse_and_restriction_consistency():
    b = W.make_config(3, n_pairs=60, ref_bases=300_000)     # tandem repeats: tie-heavy
    sc = DEFAULT
    res = oracle.align_batch(b.reads_packed, b.read_off, b.read_len, b.wins_packed, b.win_off, b.win_len,
                             b.pairs, sc, threads=4)
    for p in range(b.n_pairs):
        n, m = int(b.read_len[p]), int(b.win_len[p])
        R = W.unpack(b.reads_packed, int(b.read_off[p]), n)
        T = W.unpack(b.wins_packed, int(b.win_off[p]), m)
        s, e_ = int(res.ref_start[p]), int(res.ref_end[p])
        # P5: restricting the window to the aligned rows keeps score and CIGAR
        sub = oracle.align_pair(T[s:e_ + 1], R, sc)
        assert sub["score"] == res.score[p] and sub["cigar"] == res.cigar(p)
        # P4: reversed problem on the window prefix reaches the same score
        rev = oracle.align_pair(T[:e_ + 1][::-1], R[::-1], sc)
        assert rev["score"] == res.score[p]


# ---------------------------------------------------------------- P7 textbook special case
def test_infix_edit_distance_special_case():
    sc = OracleScoring(0, -1, 0, 1, 0.0)
    rng = random.Random(99)
    for case in range(150):
        alphabet = rng.choice(["AC", "ACGT", "ACGTN"])
        T = _rand_seq(rng, rng.randint(1, 40), alphabet)
        R = _rand_seq(rng, rng.randint(1, 25), alphabet)
        r = oracle.align_pair(T, R, sc)
        assert -r["score"] == ref.infix_edit_distance(T, R), (T, R, r)


# ---------------------------------------------------------------- degenerate shapes
def test_degenerate_shapes():
    sc = DEFAULT
    r = oracle.align_pair("A", "A", sc)
    assert (r["score"], r["ref_start"], r["ref_end"], r["cigar"]) == (1, 0, 0, "1M")
    r = oracle.align_pair("A", "C", sc)
    assert (r["score"], r["cigar"]) == (-3, "1M")
    r = oracle.align_pair("N" * 8, "ACGTACGT", sc)      # all-N window, n >= 6: all-insertion wins (R4)
    assert (r["score"], r["ref_start"], r["ref_end"], r["cigar"]) == (-(5 + 2 * 8), 1, 0, "8I")
    r = oracle.align_pair("ACG", "ACGTTTTT", sc)        # read longer than the window
    assert r["score"] == 3 - (5 + 2 * 5) and r["cigar"] == "3M5I"
    assert r["pass"] == 0
    r = oracle.align_pair("N", "N", sc)                 # N never matches, even N
    assert r["score"] == -3 and r["n_match"] == 0


def test_similarity_threshold_edges():
    # identity exactly at the threshold passes (>=), one below fails; quantised once (R12)
    T = "ACGTACGTAC"
    r = oracle.align_pair(T, "ACGTACGTAC", OracleScoring(1, -3, 5, 2, 1.0))
    assert r["pass"] == 1
    r = oracle.align_pair(T, "ACGTTCGTAC", OracleScoring(1, -3, 5, 2, 0.9))
    assert (r["n_match"], r["n_cols"], r["pass"]) == (9, 10, 1)
    r = oracle.align_pair(T, "ACGTTCGTAC", OracleScoring(1, -3, 5, 2, 0.900001))
    assert r["pass"] == 0


# ---------------------------------------------------------------- batch wrapper: packed decode with N masks on BOTH sides
def test_batch_decode_with_n_in_reads_and_windows():
    """oracle_align_batch decodes 2-bit packed reads AND windows through their N bitmaps (reading R8). The expected
    values come from the single-pair path on the original strings and, for the tiny cases, from brute force: a batch
    wrapper that drops either mask (N then decodes as 'A') fails here."""
    rng = random.Random(511)
    sc = DEFAULT
    wins, reads = [], []
    for case in range(140):                         # brute-force sized, N-rich on both sides
        wins.append(_rand_seq(rng, rng.randint(1, 6), "ACGNN"))
        reads.append(_rand_seq(rng, rng.randint(1, 5), "ACNNA"))
    for case in range(60):                          # longer, so that offsets cross word and mask-word boundaries
        wins.append(_rand_seq(rng, rng.randint(20, 90), "ACGTN"))
        reads.append(_rand_seq(rng, rng.randint(5, 40), "ACGTNA"))
    # "A" vs "N": the mask is the only thing that separates them (N is packed as code 0 = A)
    wins += ["AAAAAAAA", "NNNNNNNN", "AAAAAAAA", "ANANANAN"]
    reads += ["ANAA", "AAAA", "NNNN", "NANA"]
    b = W.batch_from_strings(wins, reads)
    assert b.read_nmask is not None and b.win_nmask is not None
    res = oracle.align_batch(b.reads_packed, b.read_off, b.read_len, b.wins_packed, b.win_off, b.win_len, b.pairs, sc,
                             read_nmask=b.read_nmask, win_nmask=b.win_nmask, threads=3)
    n_read_n_matters = 0
    for p, (T, R) in enumerate(zip(wins, reads)):
        one = oracle.align_pair(T, R, sc)
        got = dict(score=int(res.score[p]), ref_start=int(res.ref_start[p]), ref_end=int(res.ref_end[p]),
                   read_start=int(res.read_start[p]), read_end=int(res.read_end[p]), n_match=int(res.n_match[p]),
                   n_cols=int(res.n_cols[p]), cigar=res.cigar(p))
        got["pass"] = int(res.passed[p])
        for k, v in got.items():
            assert one[k] == v, (p, T, R, k, one[k], v)
        assert ref.rescore(T, R, got["ref_start"], got["cigar"], sc_tuple(sc)) == got["score"]
        if len(R) <= 5 and len(T) <= 6:
            c = ref.canonical(T, R, sc_tuple(sc))
            for k in ("score", "ref_start", "ref_end", "cigar", "n_match", "n_cols"):
                assert c[k] == got[k], (p, T, R, "bruteforce", k, c[k], got[k])
        if "N" in R and oracle.align_pair(T, R.replace("N", "A"), sc)["score"] != got["score"]:
            n_read_n_matters += 1
    assert n_read_n_matters >= 20        # the read mask really decides scores in this batch
    # hand-computed: read ANAA in AAAAAAAA is 3 matches + 1 mismatch = 0; all-N read or window: four mismatches = -12;
    # NANA against ANANANAN at offset 1 pairs N with N (mismatch) and A with A: 2 - 6 = -4
    k0 = len(wins) - 4
    assert [int(x) for x in res.score[k0:]] == [0, -12, -12, -4]
    assert [int(x) for x in res.n_match[k0:]] == [3, 0, 0, 2]
