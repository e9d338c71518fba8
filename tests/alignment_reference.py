"""Independent checkers used to pin the oracle (tests only; imports nothing from oracle/ or the
CUDA package).

* ``enumerate_all``  -- true brute force: every legal alignment of the whole read against every
  sub-region of the window, scored from its op string (a maximal gap run of k bases costs
  open + k*extend). No dynamic programming.
* ``canonical``      -- the one alignment the tie rules of DESIGN.md (readings R4-R6) select from
  the set of maximisers: lowest end row; walking backwards from the end prefer M, then D, then I,
  and inside a gap prefer to close the run (the previous op is not the same gap op) when that is
  still optimal.
* ``rescore``        -- score of a (start, CIGAR) pair against the sequences.
* ``infix_edit_distance`` -- textbook Sellers/Levenshtein DP with free window ends.
"""
from __future__ import annotations

import re
from typing import Iterator, List, Tuple


def delta(t: str, r: str, match: int, mismatch: int) -> int:
    return match if (t == r and t != "N" and r != "N") else mismatch


def score_ops(T: str, R: str, start: int, ops: str, sc) -> int:
    match, mismatch, o, e = sc
    i, j, s, k = start, 0, 0, 0
    while k < len(ops):
        op = ops[k]
        if op == "M":
            s += delta(T[i], R[j], match, mismatch)
            i += 1
            j += 1
            k += 1
        else:
            run = 0
            while k < len(ops) and ops[k] == op:
                run += 1
                k += 1
            s -= o + e * run
            if op == "I":
                j += run
            else:
                i += run
    assert j == len(R)
    return s


def enumerate_all(T: str, R: str, sc) -> Iterator[Tuple[int, int, str, int]]:
    """Yield (start, end_row, ops, score) for every legal alignment.

    start = number of window bases before the alignment; end_row = start + window bases consumed,
    restricted to 1 <= end_row <= m. No leading and no trailing D.
    """
    m, n = len(T), len(R)

    def rec(i: int, j: int, ops: List[str]):
        if j == n:
            if ops and ops[-1] != "D" and 1 <= i <= m:
                yield i, "".join(ops)
            return
        if i < m:
            ops.append("M")
            yield from rec(i + 1, j + 1, ops)
            ops.pop()
        ops.append("I")
        yield from rec(i, j + 1, ops)
        ops.pop()
        if i < m and ops:
            ops.append("D")
            yield from rec(i + 1, j, ops)
            ops.pop()

    for start in range(0, m + 1):
        for end, ops in rec(start, 0, []):
            yield start, end, ops, score_ops(T, R, start, ops, sc)


def select_canonical(cands: List[Tuple[int, str]], gap_open: int) -> Tuple[int, str]:
    """Among co-optimal (start, ops) with one common end row, apply the backward preference."""
    assert gap_open > 0, "with gap_open == 0 a run can be split for free; op strings are ambiguous"
    pool = list(cands)
    k = 1
    state = "H"
    chosen: List[str] = []
    while True:
        alive = [c for c in pool if len(c[1]) >= k]
        if not alive:
            break
        avail = {c[1][-k] for c in alive}
        if state == "H":
            order = ["M", "D", "I"]
        elif state == "D":      # just emitted D: prefer "opened here" (previous op is not D)
            order = ["M", "I", "D"]
        else:                   # just emitted I
            order = ["M", "D", "I"]
        op = next(x for x in order if x in avail)
        chosen.append(op)
        pool = [c for c in alive if c[1][-k] == op]
        state = {"M": "H", "D": "D", "I": "I"}[op]
        k += 1
    # every survivor now equals the chosen string; all read bases are consumed so lengths agree
    full = "".join(reversed(chosen))
    final = [c for c in pool if c[1] == full]
    assert final, (cands, full)
    starts = {c[0] for c in final}
    assert len(starts) == 1
    return final[0]


def canonical(T: str, R: str, sc):
    """Brute-force expected result: dict(score, ref_start, ref_end, cigar, n_match, n_cols)."""
    best = None
    pool: List[Tuple[int, int, str]] = []
    for start, end, ops, s in enumerate_all(T, R, sc):
        if best is None or s > best:
            best, pool = s, [(start, end, ops)]
        elif s == best:
            pool.append((start, end, ops))
    end = min(p[1] for p in pool)
    cands = [(p[0], p[2]) for p in pool if p[1] == end]
    out = dict(score=best, ref_end=end - 1, n_maximisers=len(pool), cands=cands)
    if sc[2] > 0:
        start, ops = select_canonical(cands, sc[2])
        i, j, nm = start, 0, 0
        for op in ops:
            if op == "M":
                nm += int(T[i] == R[j] and T[i] != "N")
                i += 1
                j += 1
            elif op == "I":
                j += 1
            else:
                i += 1
        out.update(ref_start=start, cigar=rle(ops), n_match=nm, n_cols=len(ops))
    return out


def rle(ops: str) -> str:
    out, k = [], 0
    while k < len(ops):
        r = k
        while r < len(ops) and ops[r] == ops[k]:
            r += 1
        out.append(f"{r - k}{ops[k]}")
        k = r
    return "".join(out)


def expand(cigar: str) -> str:
    return "".join(op * int(num) for num, op in re.findall(r"(\d+)([MID])", cigar))


def rescore(T: str, R: str, ref_start: int, cigar: str, sc) -> int:
    return score_ops(T, R, ref_start, expand(cigar), sc)


def infix_edit_distance(T: str, R: str) -> int:
    """min over sub-regions T' of T of the Levenshtein distance between R and T' (Sellers 1980)."""
    m, n = len(T), len(R)
    prev = [0] * (m + 1)            # zero pattern characters: free start anywhere in the text
    for j in range(1, n + 1):
        cur = [j] + [0] * m
        for i in range(1, m + 1):
            sub = prev[i - 1] + (0 if (T[i - 1] == R[j - 1] and T[i - 1] != "N") else 1)
            cur[i] = min(sub, prev[i] + 1, cur[i - 1] + 1)
        prev = cur
    return min(prev)               # free end anywhere (i = 0 allowed: costs n, never better than i >= 1 ... see test)
