"""ctypes front end of ``gotoh_oracle.c`` (TEST INFRASTRUCTURE, NOT THE PRODUCT).

The arithmetic lives in the C file, which follows PAPER.md:289-310 (recurrences and base cases),
PAPER.md:269 (result) and PAPER.md:353 (backtracking) with the tie rules listed in DESIGN.md.
This module only compiles it with gcc, marshals numpy arrays and decodes CIGAR runs.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gotoh_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None

CIGAR_OPS = "MIDNS"            # BAM op codes 0..4; the local variant emits 4 = soft clip


class _Scoring(ctypes.Structure):
    _fields_ = [("match", ctypes.c_int32), ("mismatch", ctypes.c_int32),
                ("gap_open", ctypes.c_int32), ("gap_extend", ctypes.c_int32),
                ("min_sim_q", ctypes.c_int64)]


class _Result(ctypes.Structure):
    _fields_ = [(k, ctypes.c_int32) for k in
                ("score", "ref_start", "ref_end", "read_start", "read_end", "n_match", "n_cols",
                 "pass_", "cigar_len")]


@dataclass(frozen=True)
class OracleScoring:
    match: int = 1
    mismatch: int = -3
    gap_open: int = 5
    gap_extend: int = 2
    min_similarity: float = 0.6

    def _c(self) -> _Scoring:
        # quantised once, reading R12 in DESIGN.md: q = llround(min_similarity * 1e6)
        q = int(np.floor(self.min_similarity * 1e6 + 0.5))
        return _Scoring(self.match, self.mismatch, self.gap_open, self.gap_extend, q)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    with _lock:
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
            tmp = _LIB + f".tmp{os.getpid()}"
            subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c11",
                                   "-Wall", "-o", tmp, _SRC])
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u32p, u64p, i32p, u8p = (ctypes.POINTER(t) for t in
                                 (ctypes.c_uint32, ctypes.c_uint64, ctypes.c_int32, ctypes.c_uint8))
        lib.oracle_align_pair.restype = ctypes.c_int
        lib.oracle_align_pair.argtypes = [u8p, ctypes.c_int, u8p, ctypes.c_int,
                                          ctypes.POINTER(_Scoring), ctypes.POINTER(_Result), u32p, i32p]
        lib.oracle_align_pair_local.restype = ctypes.c_int
        lib.oracle_align_pair_local.argtypes = [u8p, ctypes.c_int, u8p, ctypes.c_int,
                                                ctypes.POINTER(_Scoring), ctypes.POINTER(_Result), u32p]
        lib.oracle_align_batch_mode.restype = ctypes.c_void_p
        lib.oracle_align_batch_mode.argtypes = ([u32p, u64p, u32p, u32p] * 2 + [u32p, ctypes.c_uint64,
                                                ctypes.POINTER(_Scoring), ctypes.c_int, ctypes.c_int] +
                                                [i32p] * 5 + [u8p, i32p, i32p, u64p, u32p, i32p])
        lib.oracle_batch_n_ops.restype = ctypes.c_uint64
        lib.oracle_batch_n_ops.argtypes = [ctypes.c_void_p]
        lib.oracle_batch_fetch_ops.restype = None
        lib.oracle_batch_fetch_ops.argtypes = [ctypes.c_void_p, u32p]
        lib.oracle_batch_free.restype = None
        lib.oracle_batch_free.argtypes = [ctypes.c_void_p]
        _lib = lib
    return _lib


def _ptr(a, ctype):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ctype))


def decode_cigar(ops) -> str:
    """BAM-encoded runs ((len << 4) | op, M=0 I=1 D=2) -> '3M1D6M'."""
    return "".join(f"{int(x) >> 4}{CIGAR_OPS[int(x) & 15]}" for x in ops)


_CODE = {"A": 0, "C": 1, "G": 2, "T": 3, "N": 4}


def _codes(seq) -> np.ndarray:
    if isinstance(seq, str):
        return np.array([_CODE[c] for c in seq.upper()], dtype=np.uint8)
    return np.ascontiguousarray(seq, dtype=np.uint8)


def align_pair(window, read, scoring: OracleScoring = OracleScoring(), want_last_row: bool = False,
               local: bool = False):
    """Align one read against one window. Sequences are strings over ACGTN or code arrays.

    Returns a dict with score, ref_start, ref_end, read_start, read_end, n_match, n_cols, pass,
    cigar (string), ops (uint32 runs) and, if asked, last_row = H(i, n) for i = 0..m.
    ``local=True`` is the Smith-Waterman / soft-clipping variant (oracle_align_pair_local, R18).
    """
    lib = _load()
    T, R = _codes(window), _codes(read)
    m, n = len(T), len(R)
    if m < 1 or n < 1:
        raise ValueError("empty sequence")
    ops = np.zeros(n + m + 3, dtype=np.uint32)
    last = np.zeros(m + 1, dtype=np.int32) if want_last_row else None
    res = _Result()
    sc = scoring._c()
    if local:
        assert not want_last_row
        rc = lib.oracle_align_pair_local(_ptr(T, ctypes.c_uint8), m, _ptr(R, ctypes.c_uint8), n,
                                         ctypes.byref(sc), ctypes.byref(res), _ptr(ops, ctypes.c_uint32))
    else:
        rc = lib.oracle_align_pair(_ptr(T, ctypes.c_uint8), m, _ptr(R, ctypes.c_uint8), n,
                                   ctypes.byref(sc), ctypes.byref(res), _ptr(ops, ctypes.c_uint32),
                                   _ptr(last, ctypes.c_int32))
    if rc != 0:
        raise MemoryError("oracle_align_pair")
    ops = ops[:res.cigar_len].copy()
    out = dict(score=res.score, ref_start=res.ref_start, ref_end=res.ref_end,
               read_start=res.read_start, read_end=res.read_end, n_match=res.n_match,
               n_cols=res.n_cols, ops=ops, cigar=decode_cigar(ops))
    out["pass"] = res.pass_
    if want_last_row:
        out["last_row"] = last
    return out


@dataclass
class OracleBatchResult:
    score: np.ndarray
    ref_start: np.ndarray
    ref_end: np.ndarray
    read_start: np.ndarray
    read_end: np.ndarray
    passed: np.ndarray
    n_match: np.ndarray
    n_cols: np.ndarray
    cigar_off: np.ndarray
    cigar_len: np.ndarray
    cigar_ops: np.ndarray
    threads: int = 1

    def cigar(self, p: int) -> str:
        o, l = int(self.cigar_off[p]), int(self.cigar_len[p])
        return decode_cigar(self.cigar_ops[o:o + l])


def align_batch(reads_packed, read_off, read_len, wins_packed, win_off, win_len, pairs,
                scoring: OracleScoring = OracleScoring(), read_nmask=None, win_nmask=None,
                threads: int = 1, local: bool = False) -> OracleBatchResult:
    """Same inputs as ``sdp_align_batch`` (host numpy arrays). ``pairs`` is (P, 2) uint32."""
    lib = _load()
    reads_packed = np.ascontiguousarray(reads_packed, dtype=np.uint32)
    wins_packed = np.ascontiguousarray(wins_packed, dtype=np.uint32)
    read_off = np.ascontiguousarray(read_off, dtype=np.uint64)
    win_off = np.ascontiguousarray(win_off, dtype=np.uint64)
    read_len = np.ascontiguousarray(read_len, dtype=np.uint32)
    win_len = np.ascontiguousarray(win_len, dtype=np.uint32)
    pairs = np.ascontiguousarray(pairs, dtype=np.uint32).reshape(-1, 2)
    if read_nmask is not None:
        read_nmask = np.ascontiguousarray(read_nmask, dtype=np.uint32)
    if win_nmask is not None:
        win_nmask = np.ascontiguousarray(win_nmask, dtype=np.uint32)
    P = pairs.shape[0]
    if P and (pairs[:, 0].max() >= len(read_len) or pairs[:, 1].max() >= len(win_len)):
        raise IndexError("pair index out of range")
    i32 = lambda: np.zeros(P, dtype=np.int32)  # noqa: E731
    r = OracleBatchResult(i32(), i32(), i32(), i32(), i32(), np.zeros(P, dtype=np.uint8), i32(), i32(),
                          np.zeros(P, dtype=np.uint64), np.zeros(P, dtype=np.uint32),
                          np.zeros(0, dtype=np.uint32))
    used = ctypes.c_int32(0)
    sc = scoring._c()
    u32, u64, i32c, u8 = ctypes.c_uint32, ctypes.c_uint64, ctypes.c_int32, ctypes.c_uint8
    h = lib.oracle_align_batch_mode(
        _ptr(reads_packed, u32), _ptr(read_off, u64), _ptr(read_len, u32), _ptr(read_nmask, u32),
        _ptr(wins_packed, u32), _ptr(win_off, u64), _ptr(win_len, u32), _ptr(win_nmask, u32),
        _ptr(pairs, u32), P, ctypes.byref(sc), int(threads), 1 if local else 0,
        _ptr(r.score, i32c), _ptr(r.ref_start, i32c), _ptr(r.ref_end, i32c), _ptr(r.read_start, i32c),
        _ptr(r.read_end, i32c), _ptr(r.passed, u8), _ptr(r.n_match, i32c), _ptr(r.n_cols, i32c),
        _ptr(r.cigar_off, u64), _ptr(r.cigar_len, u32), ctypes.byref(used))
    if not h:
        raise MemoryError("oracle_align_batch")
    try:
        n_ops = lib.oracle_batch_n_ops(h)
        r.cigar_ops = np.zeros(n_ops, dtype=np.uint32)
        lib.oracle_batch_fetch_ops(h, _ptr(r.cigar_ops, u32))
    finally:
        lib.oracle_batch_free(h)
    r.threads = int(used.value)
    return r


def best_per_read(pairs: np.ndarray, score: np.ndarray, n_reads: int) -> dict:
    """Per-read choice among its candidate windows (TEST INFRASTRUCTURE, R16).

    The paper enumerates up to a ceiling of candidate regions per read and aligns the whole read to each
     but does not say how the winner is picked. Rule taken: highest score, then
    lowest window index, then lowest pair index. Written as the definition: one pass over the pairs in
    order, replacing the incumbent only when strictly better; `second_score` is the best score among the
    read's other pairs. Plain Python loop on purpose.
    """
    NO_PAIR, INT_MIN = 0xFFFFFFFF, -(2 ** 31)
    best_pair = np.full(n_reads, NO_PAIR, dtype=np.uint32)
    best_score = np.full(n_reads, INT_MIN, dtype=np.int32)
    second = np.full(n_reads, INT_MIN, dtype=np.int32)
    ncand = np.zeros(n_reads, dtype=np.uint32)
    best_win = [0] * n_reads
    for p in range(pairs.shape[0]):
        r, w, s = int(pairs[p, 0]), int(pairs[p, 1]), int(score[p])
        ncand[r] += 1
        if best_pair[r] == NO_PAIR:
            best_pair[r], best_score[r], best_win[r] = p, s, w
        elif s > best_score[r] or (s == best_score[r] and w < best_win[r]):
            second[r] = max(int(second[r]), int(best_score[r]))       # the old incumbent becomes an "other" pair
            best_pair[r], best_score[r], best_win[r] = p, s, w
        else:
            second[r] = max(int(second[r]), s)
    return dict(best_pair=best_pair, best_score=best_score, second_score=second, n_candidates=ncand)


def mate_windows(mate_pos, mate_len, mate_reverse, read_len, min_insert: int, max_insert: int, ref_bases: int):
    """Candidate region of a mate rescue (TEST INFRASTRUCTURE; R17).

    Forward-reverse orientation: a fragment is [f, f + ins) with min_insert <= ins <= max_insert; its forward end starts
    at f, its reverse end stops at f + ins. Mapped end forward at [p, p+L): the other end stops at p + ins, so it lies in
    [p + min - n, p + max). Mapped end reverse at [p, p+L): the fragment stops at p + L, the other end starts at
    p + L - ins, so it lies in [p + L - max, p + L - min + n). Clipped to the reference; length 0 when nothing is left.
    Plain Python loop on purpose."""
    off, ln = [], []
    for p, L, rev, n in zip(mate_pos, mate_len, mate_reverse, read_len):
        p, L, n = int(p), int(L), int(n)
        lo, hi = (p + min_insert - n, p + max_insert) if not rev else (p + L - max_insert, p + L - min_insert + n)
        lo, hi = max(lo, 0), min(hi, int(ref_bases))
        ok = hi > lo
        off.append(lo if ok else 0)
        ln.append(hi - lo if ok else 0)
    return np.array(off, dtype=np.uint64), np.array(ln, dtype=np.uint32)


def mate_pairs(win_len):
    """Pair list of a rescue batch (same reading): rescues whose window is not empty, in rescue order, as (k, k);
    pair_of_rescue[k] = index of rescue k in that list, 0xFFFFFFFF when its window is empty."""
    pairs, por = [], []
    for k, ln in enumerate(win_len):
        if int(ln) > 0:
            por.append(len(pairs))
            pairs.append((k, k))
        else:
            por.append(0xFFFFFFFF)
    return np.array(pairs, dtype=np.uint32).reshape(-1, 2), np.array(por, dtype=np.uint32)


def proper_pairs(mate_pos, mate_len, mate_reverse, min_insert: int, max_insert: int, win_off, win_len, ref_start, ref_end,
                 passed, pair_of_rescue=None):
    """Properly paired = aligned, passed the similarity filter, implied fragment length within the bounds (same reading).
    ref_start / ref_end / passed are indexed by pair_of_rescue[k] (rescue k itself when pair_of_rescue is None)."""
    out = []
    for k in range(len(mate_pos)):
        ok = 0
        q = k if pair_of_rescue is None else int(pair_of_rescue[k])
        if int(win_len[k]) > 0 and q != 0xFFFFFFFF and int(passed[q]):
            p, L, w = int(mate_pos[k]), int(mate_len[k]), int(win_off[k])
            ins = (w + int(ref_end[q]) + 1) - p if not mate_reverse[k] else (p + L) - (w + int(ref_start[q]))
            ok = 1 if min_insert <= ins <= max_insert else 0
        out.append(ok)
    return np.array(out, dtype=np.uint8)
