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


# ---------------------------------------------------------------- local (soft-clipping) variant, R18
def score_ops_from(T: str, R: str, i0: int, j0: int, ops: str, sc) -> int:
    """Score of an op string that starts at window base i0 and read base j0 (affine: a maximal gap run of k costs o + k e)."""
    match, mismatch, o, e = sc
    i, j, s, k = i0, j0, 0, 0
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
    return s


def enumerate_all_local(T: str, R: str, sc) -> Iterator[Tuple[int, int, int, int, str, int]]:
    """Yield (i0, j0, i_end, j_end, ops, score) for every local alignment that starts and ends with an M column:
    any window start, any read start, any end (an optimum with positive score never starts or ends in a gap when
    open + extend > 0). True brute force, no dynamic programming."""
    m, n = len(T), len(R)

    def rec(i: int, j: int, ops: List[str]):
        if ops and ops[-1] == "M":
            yield i, j, "".join(ops)
        if i < m and j < n:
            ops.append("M")
            yield from rec(i + 1, j + 1, ops)
            ops.pop()
        if ops and j < n:
            ops.append("I")
            yield from rec(i, j + 1, ops)
            ops.pop()
        if ops and i < m:
            ops.append("D")
            yield from rec(i + 1, j, ops)
            ops.pop()

    for i0 in range(m):
        for j0 in range(n):
            for ie, je, ops in rec(i0, j0, []):
                if ops[0] == "M":
                    yield i0, j0, ie, je, ops, score_ops_from(T, R, i0, j0, ops, sc)


def canonical_local(T: str, R: str, sc):
    """Brute-force expected result of the local variant: highest score; among the maximisers the lowest end row, then the
    lowest end column; walking backwards from there stop as soon as what was walked is a maximiser by itself (the DP
    cell reads 0), otherwise prefer M, then D, then I, and inside a gap prefer to close the run."""
    assert sc[2] + sc[3] > 0 and sc[2] > 0
    best, pool = 0, []
    for i0, j0, ie, je, ops, s in enumerate_all_local(T, R, sc):
        if s > best:
            best, pool = s, [(i0, j0, ie, je, ops)]
        elif s == best and s > 0:
            pool.append((i0, j0, ie, je, ops))
    n = len(R)
    if best == 0:
        return dict(score=0, ref_start=0, ref_end=-1, read_start=0, read_end=-1, cigar=f"{n}S", n_match=0, n_cols=0)
    ie = min(p[2] for p in pool)
    je = min(p[3] for p in pool if p[2] == ie)
    cands = [p for p in pool if p[2] == ie and p[3] == je]
    chosen: List[str] = []
    state = "H"
    while True:
        done = [c for c in cands if len(c[4]) == len(chosen)]
        if done and state == "H":
            final = done[0]
            break
        k = len(chosen) + 1
        alive = [c for c in cands if len(c[4]) >= k]
        avail = {c[4][-k] for c in alive}
        order = ["M", "I", "D"] if state == "D" else ["M", "D", "I"]
        op = next(x for x in order if x in avail)
        chosen.append(op)
        cands = [c for c in alive if c[4][-k] == op]
        state = {"M": "H", "D": "D", "I": "I"}[op]
    i0, j0, _, _, ops = final
    i, j, nm = i0, j0, 0
    for op in ops:
        if op == "M":
            nm += int(T[i] == R[j] and T[i] != "N")
            i += 1
            j += 1
        elif op == "I":
            j += 1
        else:
            i += 1
    cigar = (f"{j0}S" if j0 else "") + rle(ops) + (f"{n - je}S" if n - je else "")
    return dict(score=best, ref_start=i0, ref_end=ie - 1, read_start=j0, read_end=je - 1, cigar=cigar, n_match=nm,
                n_cols=len(ops), n_maximisers=len(pool))


def longest_common_substring(T: str, R: str) -> int:
    """Textbook O(mn) table of common-suffix lengths (N never matches)."""
    best = 0
    prev = [0] * (len(R) + 1)
    for i in range(1, len(T) + 1):
        cur = [0] * (len(R) + 1)
        for j in range(1, len(R) + 1):
            if T[i - 1] == R[j - 1] and T[i - 1] != "N":
                cur[j] = prev[j - 1] + 1
                best = max(best, cur[j])
        prev = cur
    return best
