"""Seeded synthetic inputs for the batched semi-global alignment path (inputs only).

This module holds none of the method's arithmetic: it produces the packed host arrays of the
C ABI (``include/sdp.h``) for the five BASELINE.json configs (recipes in DESIGN.md "Input
recipe") and packs hand-written sequences for tests. Both the CPU oracle and the CUDA path
consume its output; neither is imported here.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading
from dataclasses import dataclass, field
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_LIB = os.path.join(_HERE, "libsdpgen.so")
_lock = threading.Lock()
_lib = None

SEED_BASE = 0x13025507_0000


class _Params(ctypes.Structure):
    _fields_ = [
        ("cfg", ctypes.c_int32), ("seed", ctypes.c_uint64), ("n_pairs", ctypes.c_uint64),
        ("ref_bases", ctypes.c_uint64), ("read_len_min", ctypes.c_int32), ("read_len_max", ctypes.c_int32),
        ("win_len", ctypes.c_int32), ("win_extra", ctypes.c_int32), ("private_windows", ctypes.c_int32),
        ("random_frac", ctypes.c_double), ("sub_lo", ctypes.c_double), ("sub_hi", ctypes.c_double),
        ("indel_rate", ctypes.c_double), ("indel_geom_p", ctypes.c_double), ("indel_max", ctypes.c_int32),
        ("start_mode", ctypes.c_int32), ("start_center", ctypes.c_int32), ("start_sd", ctypes.c_double),
        ("tandem_frac", ctypes.c_double), ("divergence_mode", ctypes.c_int32),
        ("div_lo", ctypes.c_double), ("div_hi", ctypes.c_double),
    ]


def build(force: bool = False) -> str:
    with _lock:
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
            tmp = _LIB + f".tmp{os.getpid()}"
            subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c11", "-Wall",
                                   "-o", tmp, _SRC, "-lm"])
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u32p, u64p = ctypes.POINTER(ctypes.c_uint32), ctypes.POINTER(ctypes.c_uint64)
        lib.sdpgen_reference.restype = None
        lib.sdpgen_reference.argtypes = [ctypes.c_uint64, ctypes.c_uint64, u32p, u32p,
                                         ctypes.c_double, ctypes.c_double]
        lib.sdpgen_lengths.restype = None
        lib.sdpgen_lengths.argtypes = [ctypes.POINTER(_Params), u32p, u64p, u32p, u64p, u64p, u64p]
        lib.sdpgen_pairs.restype = None
        lib.sdpgen_pairs.argtypes = [ctypes.POINTER(_Params), u32p, u32p, u32p, u64p, u32p, u32p, u64p, u32p]
        _lib = lib
    return _lib


def _p(a, t):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(t))


@dataclass
class Batch:
    """Host-side arrays of one ``sdp_align_batch`` call (see include/sdp.h for the layout)."""
    reads_packed: np.ndarray
    read_off: np.ndarray
    read_len: np.ndarray
    wins_packed: np.ndarray
    win_off: np.ndarray
    win_len: np.ndarray
    pairs: np.ndarray                      # (P, 2) uint32: (read_idx, win_idx)
    read_nmask: Optional[np.ndarray] = None
    win_nmask: Optional[np.ndarray] = None
    name: str = ""
    meta: dict = field(default_factory=dict)

    @property
    def n_pairs(self) -> int:
        return int(self.pairs.shape[0])

    @property
    def cells(self) -> int:
        """Forward-matrix cells, sum over pairs of read_len * win_len (the CUPS numerator)."""
        n = self.read_len[self.pairs[:, 0]].astype(np.int64)
        m = self.win_len[self.pairs[:, 1]].astype(np.int64)
        return int((n * m).sum())

    def subset(self, idx) -> "Batch":
        """Same sequences, a subset / reordering of the pair list."""
        idx = np.asarray(idx)
        return Batch(self.reads_packed, self.read_off, self.read_len, self.wins_packed, self.win_off,
                     self.win_len, np.ascontiguousarray(self.pairs[idx]), self.read_nmask, self.win_nmask,
                     self.name + "[subset]", dict(self.meta))

    def input_bytes(self) -> int:
        tot = 0
        for a in (self.reads_packed, self.read_off, self.read_len, self.wins_packed, self.win_off,
                  self.win_len, self.pairs, self.read_nmask, self.win_nmask):
            if a is not None:
                tot += a.nbytes
        return tot


_CODE = {"A": 0, "C": 1, "G": 2, "T": 3, "N": 0}


def pack_sequences(seqs: Sequence[str], align16: bool = False):
    """Pack strings over ACGTN back to back. Returns (packed u32, off u64, len u32, nmask u32 or None)."""
    lens = np.array([len(s) for s in seqs], dtype=np.uint32)
    offs = np.zeros(len(seqs), dtype=np.uint64)
    tot = 0
    for i, s in enumerate(seqs):
        if align16:
            tot = (tot + 15) // 16 * 16
        offs[i] = tot
        tot += len(s)
    words = (tot + 15) // 16 + 4
    words = (words + 3) // 4 * 4
    packed = np.zeros(words, dtype=np.uint32)
    nmask = np.zeros((tot + 31) // 32 + 4, dtype=np.uint32)
    any_n = False
    for i, s in enumerate(seqs):
        o = int(offs[i])
        for k, c in enumerate(s.upper()):
            pos = o + k
            packed[pos >> 4] |= np.uint32(_CODE[c] << (2 * (pos & 15)))
            if c == "N":
                nmask[pos >> 5] |= np.uint32(1 << (pos & 31))
                any_n = True
    return packed, offs, lens, (nmask if any_n else None)


def batch_from_strings(windows: Sequence[str], reads: Sequence[str], pairs=None, name="strings") -> Batch:
    """Hand-written sequences -> Batch. Default pair list is (i, i)."""
    rp, ro, rl, rn = pack_sequences(reads)
    wp, wo, wl, wn = pack_sequences(windows)
    if pairs is None:
        assert len(windows) == len(reads)
        pairs = np.stack([np.arange(len(reads))] * 2, axis=1)
    pairs = np.ascontiguousarray(pairs, dtype=np.uint32).reshape(-1, 2)
    return Batch(rp, ro, rl, wp, wo, wl, pairs, rn, wn, name)


def unpack(packed: np.ndarray, off: int, length: int, nmask: Optional[np.ndarray] = None) -> str:
    """Decode one sequence back to a string (for error messages and tests)."""
    out = []
    for k in range(off, off + length):
        if nmask is not None and (int(nmask[k >> 5]) >> (k & 31)) & 1:
            out.append("N")
        else:
            out.append("ACGT"[(int(packed[k >> 4]) >> (2 * (k & 15))) & 3])
    return "".join(out)


# BASELINE.json configs -> generator parameters
_FULL = {
    1: dict(n_pairs=1_000, ref_bases=1_000_000),
    2: dict(n_pairs=1_000_000, ref_bases=100_000_000),
    3: dict(n_pairs=2_000_000, ref_bases=100_000_000),
    4: dict(n_pairs=500_000, ref_bases=100_000_000),
    5: dict(n_pairs=4_000_000, ref_bases=100_000_000),
}


def _params(cfg: int, n_pairs: int, ref_bases: int, seed: int) -> _Params:
    P = _Params()
    P.cfg, P.seed, P.n_pairs, P.ref_bases = cfg, seed, n_pairs, ref_bases
    P.win_extra = 0
    P.private_windows = 0
    P.tandem_frac = 0.0
    P.divergence_mode = 0
    P.start_mode = 0
    if cfg == 1:
        P.read_len_min = P.read_len_max = 100
        P.win_len = 300
        P.random_frac, P.sub_lo, P.sub_hi, P.indel_rate = 0.10, 0.02, 0.02, 0.003
        P.indel_geom_p, P.indel_max = 0.5, 10
    elif cfg == 2:
        P.read_len_min = P.read_len_max = 100
        P.win_len = 500
        P.random_frac, P.sub_lo, P.sub_hi, P.indel_rate = 0.05, 0.01, 0.01, 0.002
        P.indel_geom_p, P.indel_max = 0.5, 10
        P.start_mode, P.start_center, P.start_sd = 1, 200, 50.0
    elif cfg == 3:
        P.read_len_min = P.read_len_max = 150
        P.win_len = 600
        P.private_windows = 1
        P.random_frac, P.sub_lo, P.sub_hi, P.indel_rate = 0.0, 0.005, 0.03, 0.003
        P.indel_geom_p, P.indel_max = 0.25, 20
        P.tandem_frac = 0.20
    elif cfg == 4:
        P.read_len_min = P.read_len_max = 250
        P.win_len = 750
        P.random_frac = 0.0
        P.divergence_mode, P.div_lo, P.div_hi = 1, 0.10, 0.40
        P.indel_geom_p, P.indel_max = 0.0, 30
    elif cfg == 5:
        P.read_len_min, P.read_len_max = 50, 300
        P.win_len, P.win_extra = 0, 300
        P.random_frac, P.sub_lo, P.sub_hi, P.indel_rate = 0.05, 0.015, 0.015, 0.003
        P.indel_geom_p, P.indel_max = 0.5, 10
        P.start_mode, P.start_center, P.start_sd = 1, 150, 50.0
    else:
        raise ValueError(f"unknown config {cfg}")
    return P


_ref_cache: dict = {}


def reference(ref_bases: int, seed: int, with_n: bool):
    """Packed i.i.d. uniform reference (+ N-run mask for config 5), cached per (size, seed, N)."""
    key = (ref_bases, seed, with_n)
    if key not in _ref_cache:
        lib = _load()
        words = ((ref_bases + 15) // 16 + 4 + 3) // 4 * 4
        packed = np.zeros(words, dtype=np.uint32)
        nmask = np.zeros(((ref_bases + 31) // 32 + 4 + 3) // 4 * 4, dtype=np.uint32) if with_n else None
        lib.sdpgen_reference(seed, ref_bases, _p(packed, ctypes.c_uint32), _p(nmask, ctypes.c_uint32),
                             4500.0, 500.0)
        if len(_ref_cache) > 4:
            _ref_cache.clear()
        _ref_cache[key] = (packed, nmask)
    return _ref_cache[key]


def make_config(cfg: int, n_pairs: Optional[int] = None, ref_bases: Optional[int] = None,
                seed: Optional[int] = None) -> Batch:
    """One of the five BASELINE.json workloads; ``n_pairs`` / ``ref_bases`` shrink it for tests."""
    full = _FULL[cfg]
    n_pairs = full["n_pairs"] if n_pairs is None else int(n_pairs)
    ref_bases = full["ref_bases"] if ref_bases is None else int(ref_bases)
    seed = SEED_BASE + cfg if seed is None else int(seed)
    # configs 2-5 share one 100 Mbp reference (seed of config 2); config 5 adds the N-run mask
    ref_seed = SEED_BASE + (1 if cfg == 1 else 2)
    ref_packed, ref_nmask = reference(ref_bases, ref_seed, with_n=(cfg == 5))
    P = _params(cfg, n_pairs, ref_bases, seed)
    return _generate(P, ref_packed, ref_nmask, name=f"cfg{cfg}",
                     meta=dict(cfg=cfg, n_pairs=n_pairs, ref_bases=ref_bases, seed=seed))


def make_long_reads(n_pairs: int, read_len: int, win_len: int, ref_bases: Optional[int] = None,
                    seed: Optional[int] = None) -> Batch:
    """Config 2's recipe (mate-rescue shape: 5 % unrelated reads, 1 % substitutions, indels at 0.2 % per base, true
    start normal around the window's middle) at another read and window length: the long-read case of PAPER.md:117
    ("read length is not capped"). Windows are views into the shared seeded reference."""
    ref_bases = _FULL[2]["ref_bases"] if ref_bases is None else int(ref_bases)
    seed = SEED_BASE + 900 + read_len if seed is None else int(seed)
    ref_packed, ref_nmask = reference(ref_bases, SEED_BASE + 2, with_n=False)
    P = _params(2, int(n_pairs), ref_bases, seed)
    P.read_len_min = P.read_len_max = int(read_len)
    P.win_len = int(win_len)
    P.start_center, P.start_sd = max(0, (int(win_len) - int(read_len)) // 2), max(1.0, (win_len - read_len) / 8.0)
    return _generate(P, ref_packed, ref_nmask, name=f"long{read_len}x{win_len}",
                     meta=dict(n_pairs=int(n_pairs), read_len=int(read_len), win_len=int(win_len), ref_bases=ref_bases,
                               seed=seed))


def _generate(P: _Params, ref_packed, ref_nmask, name: str, meta: dict) -> Batch:
    lib = _load()
    n_pairs = int(P.n_pairs)
    read_len = np.zeros(n_pairs, dtype=np.uint32)
    read_off = np.zeros(n_pairs, dtype=np.uint64)
    win_len = np.zeros(n_pairs, dtype=np.uint32)
    win_off = np.zeros(n_pairs, dtype=np.uint64)
    tr, tw = ctypes.c_uint64(0), ctypes.c_uint64(0)
    lib.sdpgen_lengths(ctypes.byref(P), _p(read_len, ctypes.c_uint32), _p(read_off, ctypes.c_uint64),
                       _p(win_len, ctypes.c_uint32),
                       _p(win_off, ctypes.c_uint64) if P.private_windows else None,
                       ctypes.byref(tr), ctypes.byref(tw))
    reads_packed = np.zeros(((tr.value + 15) // 16 + 4 + 3) // 4 * 4, dtype=np.uint32)
    wins_out = (np.zeros(((tw.value + 15) // 16 + 4 + 3) // 4 * 4, dtype=np.uint32)
                if P.private_windows else None)
    lib.sdpgen_pairs(ctypes.byref(P), _p(ref_packed, ctypes.c_uint32), _p(ref_nmask, ctypes.c_uint32),
                     _p(read_len, ctypes.c_uint32), _p(read_off, ctypes.c_uint64),
                     _p(reads_packed, ctypes.c_uint32), _p(win_len, ctypes.c_uint32),
                     _p(win_off, ctypes.c_uint64), _p(wins_out, ctypes.c_uint32))
    idx = np.arange(n_pairs, dtype=np.uint32)
    pairs = np.ascontiguousarray(np.stack([idx, idx], axis=1))
    return Batch(reads_packed, read_off, read_len,
                 wins_out if P.private_windows else ref_packed, win_off, win_len, pairs,
                 None, None if P.private_windows else ref_nmask, name=name, meta=meta)


def make_step3(n_reads: int, max_candidates: int = 30, ref_bases: Optional[int] = None,
               seed: Optional[int] = None) -> Batch:
    """Step-3 shape: each read against up to ``max_candidates`` candidate windows.

    Reads and their true windows come from the config-2 generator (100 bp reads, 500 bp windows cut from
    the seeded reference). Every read gets c ~ U{1..max_candidates} candidates: its true window, up to two
    windows shifted by +-U{20..150} bases (overlapping the true locus, so scores tie or nearly tie), and
    uniformly placed decoys. Windows are views into the packed reference; the pair list is grouped by read
    with the candidates of a read in random order. No alignment arithmetic here.
    """
    base = make_config(2, n_pairs=n_reads, ref_bases=ref_bases, seed=seed)
    rng = np.random.default_rng(SEED_BASE + 77 if seed is None else int(seed) + 77)
    ref_len = int(base.wins_packed.shape[0]) * 16 - 64
    m = int(base.win_len[0])
    ncand = rng.integers(1, max_candidates + 1, size=n_reads)
    total = int(ncand.sum())
    read_idx = np.repeat(np.arange(n_reads, dtype=np.uint32), ncand)
    first = np.concatenate([[0], np.cumsum(ncand)[:-1]])
    slot = np.arange(total) - np.repeat(first, ncand)            # 0 = true window, 1..2 = shifted, rest decoys
    true_off = base.win_off[read_idx].astype(np.int64)
    shift = rng.integers(20, 151, size=total) * rng.choice([-1, 1], size=total)
    decoy = rng.integers(0, max(1, ref_len - m), size=total)
    off = np.where(slot == 0, true_off, np.where(slot <= 2, true_off + shift, decoy))
    off = np.clip(off, 0, max(0, ref_len - m)).astype(np.uint64)
    order = np.lexsort((rng.random(total), read_idx))            # shuffle inside each read's group
    win_off = np.ascontiguousarray(off[order])
    pairs = np.ascontiguousarray(np.stack([read_idx[order], np.arange(total, dtype=np.uint32)], axis=1))
    return Batch(base.reads_packed, base.read_off, base.read_len, base.wins_packed, win_off,
                 np.full(total, m, dtype=np.uint32), pairs, base.read_nmask, base.win_nmask,
                 f"step3[{n_reads} reads x <= {max_candidates}]", dict(base.meta))
