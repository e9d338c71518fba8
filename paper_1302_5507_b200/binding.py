"""Thin ctypes binding of libsdp.so (include/sdp.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI. PyTorch appears here only as
the owner of device memory and streams (``torch.Tensor.data_ptr()``, ``torch.cuda.Stream``).
There is no CPU fallback: loading fails loudly if the library is missing.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsdp.so")

SDP_OK, SDP_EINVAL, SDP_ERANGE, SDP_ECUDA, SDP_ENOMEM = 0, -1, -2, -3, -4
SDP_MAX_READ_LEN = 1024
SDP_MAX_SEQ_LEN = 1000000
SDP_MAX_CELL_VALUE = 32000
SDP_ROUTE_NO_THIN, SDP_ROUTE_NO_WIDE, SDP_ROUTE_ALWAYS_REVERSE = 1, 2, 4

EXPORTS = ["sdp_create", "sdp_align_batch", "sdp_align_batch_host", "sdp_get_stats", "sdp_set_timing",
           "sdp_last_error", "sdp_destroy", "sdp_measure_dpx_rate", "sdp_version", "sdp_best_per_read",
           "sdp_set_score_only", "sdp_set_prefilter", "sdp_set_debug_route", "sdp_set_mode", "sdp_set_chunks", "sdp_mate_windows", "sdp_mate_pairs",
           "sdp_proper_pairs", "sdp_best_per_read_static", "sdp_static_last_error"]


class SdpError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"sdp error {code}: {msg}")
        self.code = code


class sdp_scoring(ctypes.Structure):
    _fields_ = [("match", ctypes.c_int32), ("mismatch", ctypes.c_int32), ("gap_open", ctypes.c_int32),
                ("gap_extend", ctypes.c_int32), ("min_similarity", ctypes.c_double)]


class sdp_batch(ctypes.Structure):
    _fields_ = [("reads_packed", ctypes.c_void_p), ("read_off", ctypes.c_void_p), ("read_len", ctypes.c_void_p),
                ("read_nmask", ctypes.c_void_p), ("n_reads", ctypes.c_uint32), ("reads_bases", ctypes.c_uint64),
                ("wins_packed", ctypes.c_void_p), ("win_off", ctypes.c_void_p), ("win_len", ctypes.c_void_p),
                ("win_nmask", ctypes.c_void_p), ("n_wins", ctypes.c_uint32), ("wins_bases", ctypes.c_uint64),
                ("pairs", ctypes.c_void_p), ("n_pairs", ctypes.c_uint64)]


class sdp_result(ctypes.Structure):
    _fields_ = [("score", ctypes.c_void_p), ("ref_start", ctypes.c_void_p), ("ref_end", ctypes.c_void_p),
                ("read_start", ctypes.c_void_p), ("read_end", ctypes.c_void_p), ("pass_", ctypes.c_void_p),
                ("n_match", ctypes.c_void_p), ("n_cols", ctypes.c_void_p), ("cigar_off", ctypes.c_void_p),
                ("cigar_len", ctypes.c_void_p), ("cigar_ops", ctypes.c_void_p), ("n_cigar_ops", ctypes.c_uint64),
                ("n_pairs", ctypes.c_uint64)]


class sdp_read_best(ctypes.Structure):
    _fields_ = [("best_pair", ctypes.c_void_p), ("best_score", ctypes.c_void_p), ("second_score", ctypes.c_void_p),
                ("n_candidates", ctypes.c_void_p), ("n_reads", ctypes.c_uint32)]


class sdp_mates(ctypes.Structure):
    _fields_ = [("mate_pos", ctypes.c_void_p), ("mate_len", ctypes.c_void_p), ("mate_reverse", ctypes.c_void_p),
                ("read_len", ctypes.c_void_p), ("n", ctypes.c_uint64)]


SDP_NO_PAIR = 0xFFFFFFFF


class sdp_stats(ctypes.Structure):
    _fields_ = [("n_pairs", ctypes.c_uint64), ("cells_forward", ctypes.c_uint64), ("cells_reverse", ctypes.c_uint64),
                ("cells_traceback", ctypes.c_uint64), ("n_reverse_pairs", ctypes.c_uint64),
                ("kernel_launches", ctypes.c_uint32), ("forward_launches", ctypes.c_uint32),
                ("ms_total", ctypes.c_float), ("ms_bucket", ctypes.c_float), ("ms_forward", ctypes.c_float),
                ("ms_reverse", ctypes.c_float), ("ms_traceback", ctypes.c_float), ("ms_compact", ctypes.c_float),
                ("cells_prefiltered", ctypes.c_uint64), ("n_slow_words", ctypes.c_uint64)]

    def as_dict(self) -> dict:
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def load_library(path: Optional[str] = None) -> ctypes.CDLL:
    """dlopen libsdp.so and declare the prototypes. Raises if the library was not built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or LIB_PATH
    if not os.path.exists(path):
        raise FileNotFoundError(f"{path} not found: build it with `python -m paper_1302_5507_b200.build` "
                                "(the CUDA library is the product; there is no CPU fallback)")
    lib = ctypes.CDLL(path)
    lib.sdp_create.restype = ctypes.c_int
    lib.sdp_create.argtypes = [ctypes.POINTER(sdp_scoring), ctypes.c_int, ctypes.POINTER(ctypes.c_void_p)]
    lib.sdp_align_batch.restype = ctypes.c_int
    lib.sdp_align_batch.argtypes = [ctypes.c_void_p, ctypes.POINTER(sdp_batch), ctypes.c_void_p,
                                    ctypes.POINTER(sdp_result)]
    lib.sdp_align_batch_host.restype = ctypes.c_int
    lib.sdp_align_batch_host.argtypes = [ctypes.c_void_p, ctypes.POINTER(sdp_batch), ctypes.POINTER(sdp_result)]
    lib.sdp_best_per_read.restype = ctypes.c_int
    lib.sdp_best_per_read.argtypes = [ctypes.c_void_p, ctypes.POINTER(sdp_batch), ctypes.POINTER(sdp_result),
                                      ctypes.c_void_p, ctypes.POINTER(sdp_read_best)]
    lib.sdp_best_per_read_static.restype = ctypes.c_int
    lib.sdp_best_per_read_static.argtypes = [ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint32,
                                             ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    lib.sdp_static_last_error.restype = ctypes.c_char_p
    lib.sdp_static_last_error.argtypes = []
    lib.sdp_mate_windows.restype = ctypes.c_int
    lib.sdp_mate_windows.argtypes = [ctypes.c_void_p, ctypes.POINTER(sdp_mates), ctypes.c_uint32, ctypes.c_uint32,
                                     ctypes.c_uint64, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    lib.sdp_proper_pairs.restype = ctypes.c_int
    lib.sdp_proper_pairs.argtypes = [ctypes.c_void_p, ctypes.POINTER(sdp_mates), ctypes.c_uint32, ctypes.c_uint32,
                                     ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                     ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    lib.sdp_mate_pairs.restype = ctypes.c_int
    lib.sdp_mate_pairs.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_void_p, ctypes.c_void_p,
                                   ctypes.c_void_p, ctypes.POINTER(ctypes.c_uint64)]
    lib.sdp_set_prefilter.restype = ctypes.c_int
    lib.sdp_set_prefilter.argtypes = [ctypes.c_void_p, ctypes.c_int]
    lib.sdp_set_debug_route.restype = ctypes.c_int
    lib.sdp_set_debug_route.argtypes = [ctypes.c_void_p, ctypes.c_uint32]
    lib.sdp_set_mode.restype = ctypes.c_int
    lib.sdp_set_mode.argtypes = [ctypes.c_void_p, ctypes.c_int]
    lib.sdp_set_score_only.restype = ctypes.c_int
    lib.sdp_set_score_only.argtypes = [ctypes.c_void_p, ctypes.c_int]
    lib.sdp_set_chunks.restype = ctypes.c_int
    lib.sdp_set_chunks.argtypes = [ctypes.c_void_p, ctypes.c_int]
    lib.sdp_get_stats.restype = ctypes.c_int
    lib.sdp_get_stats.argtypes = [ctypes.c_void_p, ctypes.POINTER(sdp_stats)]
    lib.sdp_set_timing.restype = ctypes.c_int
    lib.sdp_set_timing.argtypes = [ctypes.c_void_p, ctypes.c_int]
    lib.sdp_last_error.restype = ctypes.c_char_p
    lib.sdp_last_error.argtypes = [ctypes.c_void_p]
    lib.sdp_destroy.restype = None
    lib.sdp_destroy.argtypes = [ctypes.c_void_p]
    lib.sdp_measure_dpx_rate.restype = ctypes.c_int
    lib.sdp_measure_dpx_rate.argtypes = [ctypes.c_int, ctypes.POINTER(ctypes.c_double),
                                         ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_double)]
    lib.sdp_version.restype = ctypes.c_char_p
    lib.sdp_version.argtypes = []
    _lib = lib
    return lib


def sdp_version() -> str:
    return load_library().sdp_version().decode()


def sdp_measure_dpx_rate(device: int = 0) -> dict:
    rate, sms, mhz = ctypes.c_double(0), ctypes.c_int32(0), ctypes.c_double(0)
    rc = load_library().sdp_measure_dpx_rate(device, ctypes.byref(rate), ctypes.byref(sms), ctypes.byref(mhz))
    if rc != SDP_OK:
        raise SdpError(rc, "sdp_measure_dpx_rate")
    return dict(instr_per_clk_per_sm=rate.value, sm_count=sms.value, sm_mhz=mhz.value)


SDP_STATIC_MAX_READS = 1 << 20


def best_per_read_static(pairs, score, n_pairs: int, n_reads: int, best_pair, best_score, second_score, n_candidates,
                         device: int = 0, stream=None) -> None:
    """sdp_best_per_read_static: the per-read choice without a context and without any device allocation by the
    library, for callers whose GPU memory is all spoken for. Every array is device memory the caller made beforehand,
    given as a torch CUDA tensor or a raw device address (e.g. ``sdp_result.score``): ``pairs`` (int32 [n_pairs, 2])
    and ``score`` (int32 [n_pairs]) in, the four int32 [n_reads] arrays out (best_pair and n_candidates hold unsigned
    values). Only enqueues on ``stream`` (default: torch's current stream): synchronise before reading. Raises
    SdpError, e.g. SDP_ERANGE when n_reads > SDP_STATIC_MAX_READS."""
    import torch
    if stream is None:
        stream = torch.cuda.current_stream(device)

    def ptr(x):
        return ctypes.c_void_p(x.data_ptr() if hasattr(x, "data_ptr") else x)

    lib = load_library()
    rc = lib.sdp_best_per_read_static(device, ptr(pairs), ptr(score), int(n_pairs), int(n_reads),
                                      ctypes.c_void_p(stream.cuda_stream), ptr(best_pair), ptr(best_score),
                                      ptr(second_score), ptr(n_candidates))
    if rc != SDP_OK:
        raise SdpError(rc, lib.sdp_static_last_error().decode())


@dataclass
class DeviceBatch:
    """Inputs of one call resident in HBM (torch tensors keep the memory alive)."""
    tensors: dict
    c: sdp_batch
    n_pairs: int


@dataclass
class HostResult:
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

    def cigar(self, p: int) -> str:
        o, l = int(self.cigar_off[p]), int(self.cigar_len[p])
        return "".join(f"{int(x) >> 4}{'MIDNS'[int(x) & 15]}" for x in self.cigar_ops[o:o + l])


_cudart_lib = None


def _cudart():
    """The CUDA runtime torch already loaded (used only to read results back in tests)."""
    global _cudart_lib
    if _cudart_lib is None:
        import glob
        import torch
        cands = ["libcudart.so.12", "libcudart.so"]
        cands += glob.glob(os.path.join(os.path.dirname(torch.__file__), "lib", "libcudart*.so*"))
        cands += glob.glob(os.path.join(os.path.dirname(os.path.dirname(torch.__file__)),
                                        "nvidia", "cuda_runtime", "lib", "libcudart.so*"))
        cands += glob.glob("/usr/local/cuda/lib64/libcudart.so*")
        for c in cands:
            try:
                _cudart_lib = ctypes.CDLL(c)
                break
            except OSError:
                continue
        if _cudart_lib is None:
            raise SdpError(SDP_ECUDA, "libcudart not found")
        _cudart_lib.cudaMemcpy.restype = ctypes.c_int
    return _cudart_lib


def _np_view(ptr: int, n: int, dtype) -> np.ndarray:
    if n == 0:
        return np.zeros(0, dtype=dtype)
    nbytes = n * np.dtype(dtype).itemsize
    buf = (ctypes.c_char * nbytes).from_address(ptr)
    return np.frombuffer(buf, dtype=dtype, count=n)


class Context:
    """sdp_create / sdp_align_batch / sdp_destroy with the same names and argument meaning."""

    def __init__(self, match: int = 1, mismatch: int = -3, gap_open: int = 5, gap_extend: int = 2,
                 min_similarity: float = 0.6, device: int = 0):
        self._lib = load_library()
        self._h = ctypes.c_void_p()
        sc = sdp_scoring(match, mismatch, gap_open, gap_extend, min_similarity)
        rc = self._lib.sdp_create(ctypes.byref(sc), device, ctypes.byref(self._h))
        if rc != SDP_OK:
            self._h = ctypes.c_void_p()
            raise SdpError(rc, "sdp_create failed (bad scoring, bad device, or CUDA unavailable)")
        self.device = device

    # -- lifetime
    def destroy(self):
        if self._h:
            self._lib.sdp_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.destroy()

    def last_error(self) -> str:
        return self._lib.sdp_last_error(self._h).decode()

    def set_timing(self, enabled: bool):
        self._lib.sdp_set_timing(self._h, int(bool(enabled)))

    def set_prefilter(self, enabled: bool):
        self._lib.sdp_set_prefilter(self._h, int(bool(enabled)))

    def set_debug_route(self, no_thin: bool = False, no_wide: bool = False, force_g: int = 0, always_reverse: bool = False):
        """sdp_set_debug_route: route pairs through the other traceback kernels / force a thread-group size (tests)."""
        flags = ((SDP_ROUTE_NO_THIN if no_thin else 0) | (SDP_ROUTE_NO_WIDE if no_wide else 0) |
                 (SDP_ROUTE_ALWAYS_REVERSE if always_reverse else 0) | ((int(force_g) & 0x3F) << 8))
        self._check(self._lib.sdp_set_debug_route(self._h, flags))

    def set_mode(self, local: bool):
        """sdp_set_mode: False = the paper's semi-global formulation (default), True = local / soft-clipping variant."""
        self._check(self._lib.sdp_set_mode(self._h, 1 if local else 0))

    def set_chunks(self, chunks: int):
        """sdp_set_chunks: lanes one call's pair list is split into (0 = automatic, 1 = no pipelining)."""
        self._check(self._lib.sdp_set_chunks(self._h, int(chunks)))

    def set_score_only(self, enabled: bool):
        self._lib.sdp_set_score_only(self._h, int(bool(enabled)))

    def stats(self) -> dict:
        s = sdp_stats()
        self._lib.sdp_get_stats(self._h, ctypes.byref(s))
        return s.as_dict()

    def _check(self, rc: int):
        if rc != SDP_OK:
            raise SdpError(rc, self.last_error())

    # -- device path
    def upload(self, batch) -> DeviceBatch:
        """Copy a workloads.Batch (host numpy arrays) into HBM as torch tensors."""
        import torch
        dev = torch.device("cuda", self.device)

        def up(a, dtype):
            if a is None:
                return None
            a = np.ascontiguousarray(a)
            return torch.from_numpy(a.view(dtype)).to(dev)

        t = dict(reads_packed=up(batch.reads_packed, np.int32), read_off=up(batch.read_off, np.int64),
                 read_len=up(batch.read_len, np.int32), read_nmask=up(batch.read_nmask, np.int32),
                 wins_packed=up(batch.wins_packed, np.int32), win_off=up(batch.win_off, np.int64),
                 win_len=up(batch.win_len, np.int32), win_nmask=up(batch.win_nmask, np.int32),
                 pairs=up(batch.pairs.reshape(-1), np.int32))
        c = self._c_batch({k: (v.data_ptr() if v is not None else None) for k, v in t.items()}, batch)
        return DeviceBatch(t, c, batch.n_pairs)

    @staticmethod
    def _c_batch(ptrs: dict, batch) -> sdp_batch:
        return sdp_batch(ptrs["reads_packed"], ptrs["read_off"], ptrs["read_len"], ptrs["read_nmask"],
                         len(batch.read_len), len(batch.reads_packed) * 16,
                         ptrs["wins_packed"], ptrs["win_off"], ptrs["win_len"], ptrs["win_nmask"],
                         len(batch.win_len), len(batch.wins_packed) * 16,
                         ptrs["pairs"], batch.n_pairs)

    def align_batch(self, dbatch: DeviceBatch, stream=None) -> sdp_result:
        """sdp_align_batch on device-resident inputs; returns the raw result (device pointers)."""
        import torch
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        res = sdp_result()
        self._check(self._lib.sdp_align_batch(self._h, ctypes.byref(dbatch.c), ctypes.c_void_p(stream.cuda_stream),
                                              ctypes.byref(res)))
        return res

    def fetch(self, res: sdp_result) -> HostResult:
        """Copy a device-side sdp_result to host numpy arrays (test / inspection helper)."""
        P, n_ops = int(res.n_pairs), int(res.n_cigar_ops)
        cudart = _cudart()

        def down(ptr, n, dtype):
            out = np.zeros(n, dtype=dtype)
            if n:
                err = cudart.cudaMemcpy(ctypes.c_void_p(out.ctypes.data), ctypes.c_void_p(ptr),
                                        ctypes.c_size_t(out.nbytes), 2)   # cudaMemcpyDeviceToHost
                if int(err) != 0:
                    raise SdpError(SDP_ECUDA, f"cudaMemcpy D2H failed: {err}")
            return out

        return HostResult(down(res.score, P, np.int32), down(res.ref_start, P, np.int32),
                          down(res.ref_end, P, np.int32), down(res.read_start, P, np.int32),
                          down(res.read_end, P, np.int32), down(res.pass_, P, np.uint8),
                          down(res.n_match, P, np.int32), down(res.n_cols, P, np.int32),
                          down(res.cigar_off, P, np.uint64), down(res.cigar_len, P, np.uint32),
                          down(res.cigar_ops, n_ops, np.uint32))

    def best_per_read(self, dbatch: DeviceBatch, res: sdp_result, stream=None) -> dict:
        """sdp_best_per_read on the result of the last align_batch; returns host numpy arrays."""
        import torch
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        rb = sdp_read_best()
        self._check(self._lib.sdp_best_per_read(self._h, ctypes.byref(dbatch.c), ctypes.byref(res),
                                                ctypes.c_void_p(stream.cuda_stream), ctypes.byref(rb)))
        cudart, R = _cudart(), int(rb.n_reads)

        def down(ptr, dtype):
            out = np.zeros(R, dtype=dtype)
            if R and int(cudart.cudaMemcpy(ctypes.c_void_p(out.ctypes.data), ctypes.c_void_p(ptr),
                                           ctypes.c_size_t(out.nbytes), 2)) != 0:
                raise SdpError(SDP_ECUDA, "cudaMemcpy D2H failed")
            return out

        return dict(best_pair=down(rb.best_pair, np.uint32), best_score=down(rb.best_score, np.int32),
                    second_score=down(rb.second_score, np.int32), n_candidates=down(rb.n_candidates, np.uint32))

    # -- mate rescue (device tensors in, device tensors out; argument marshalling only)
    @staticmethod
    def _mates(mate_pos, mate_len, mate_reverse, read_len) -> sdp_mates:
        return sdp_mates(mate_pos.data_ptr(), mate_len.data_ptr(), mate_reverse.data_ptr(), read_len.data_ptr(),
                         int(mate_pos.numel()))

    def mate_windows(self, mate_pos, mate_len, mate_reverse, read_len, min_insert: int, max_insert: int, ref_bases: int):
        """sdp_mate_windows: torch CUDA tensors (int64 / int32 / uint8 / int32) -> (win_off int64, win_len int32) tensors."""
        import torch
        n = int(mate_pos.numel())
        win_off = torch.empty(n, dtype=torch.int64, device=mate_pos.device)
        win_len = torch.empty(n, dtype=torch.int32, device=mate_pos.device)
        m = self._mates(mate_pos, mate_len, mate_reverse, read_len)
        st = torch.cuda.current_stream(self.device)
        self._check(self._lib.sdp_mate_windows(self._h, ctypes.byref(m), int(min_insert), int(max_insert), int(ref_bases),
                                               ctypes.c_void_p(st.cuda_stream), ctypes.c_void_p(win_off.data_ptr()),
                                               ctypes.c_void_p(win_len.data_ptr())))
        return win_off, win_len

    def mate_pairs(self, win_len):
        """sdp_mate_pairs: win_len CUDA tensor -> (pairs (P, 2) int32 CUDA tensor, pair_of_rescue int32 CUDA tensor)."""
        import torch
        n = int(win_len.numel())
        pairs = torch.empty(max(2 * n, 1), dtype=torch.int32, device=win_len.device)
        por = torch.empty(max(n, 1), dtype=torch.int32, device=win_len.device)
        cnt = ctypes.c_uint64(0)
        st = torch.cuda.current_stream(self.device)
        self._check(self._lib.sdp_mate_pairs(self._h, ctypes.c_void_p(win_len.data_ptr()), n, ctypes.c_void_p(st.cuda_stream),
                                             ctypes.c_void_p(pairs.data_ptr()), ctypes.c_void_p(por.data_ptr()),
                                             ctypes.byref(cnt)))
        return pairs[:2 * int(cnt.value)].reshape(-1, 2), por[:n]

    def proper_pairs(self, mate_pos, mate_len, mate_reverse, read_len, min_insert: int, max_insert: int, win_off, win_len,
                     res: sdp_result, pair_of_rescue=None):
        """sdp_proper_pairs on the sdp_result of aligning the rescue batch; returns a uint8 CUDA tensor."""
        import torch
        n = int(mate_pos.numel())
        proper = torch.empty(n, dtype=torch.uint8, device=mate_pos.device)
        m = self._mates(mate_pos, mate_len, mate_reverse, read_len)
        st = torch.cuda.current_stream(self.device)
        self._check(self._lib.sdp_proper_pairs(self._h, ctypes.byref(m), int(min_insert), int(max_insert),
                                               ctypes.c_void_p(win_off.data_ptr()), ctypes.c_void_p(win_len.data_ptr()),
                                               ctypes.c_void_p(pair_of_rescue.data_ptr()) if pair_of_rescue is not None else None,
                                               ctypes.c_void_p(res.ref_start), ctypes.c_void_p(res.ref_end),
                                               ctypes.c_void_p(res.pass_), ctypes.c_void_p(st.cuda_stream),
                                               ctypes.c_void_p(proper.data_ptr())))
        return proper

    # -- host path
    def align_batch_host(self, batch) -> HostResult:
        """sdp_align_batch_host: host arrays in, host arrays out (copies happen inside the call)."""
        keep = {}

        def ptr(a):
            if a is None:
                return None
            a = np.ascontiguousarray(a)
            keep[id(a)] = a
            return a.ctypes.data

        c = self._c_batch(dict(reads_packed=ptr(batch.reads_packed), read_off=ptr(batch.read_off),
                               read_len=ptr(batch.read_len), read_nmask=ptr(batch.read_nmask),
                               wins_packed=ptr(batch.wins_packed), win_off=ptr(batch.win_off),
                               win_len=ptr(batch.win_len), win_nmask=ptr(batch.win_nmask),
                               pairs=ptr(batch.pairs)), batch)
        res = sdp_result()
        self._check(self._lib.sdp_align_batch_host(self._h, ctypes.byref(c), ctypes.byref(res)))
        P, n_ops = int(res.n_pairs), int(res.n_cigar_ops)
        v = lambda p, n, dt: _np_view(p, n, dt).copy()  # noqa: E731  (ctx-owned pinned memory -> caller copy)
        return HostResult(v(res.score, P, np.int32), v(res.ref_start, P, np.int32), v(res.ref_end, P, np.int32),
                          v(res.read_start, P, np.int32), v(res.read_end, P, np.int32), v(res.pass_, P, np.uint8),
                          v(res.n_match, P, np.int32), v(res.n_cols, P, np.int32), v(res.cigar_off, P, np.uint64),
                          v(res.cigar_len, P, np.uint32), v(res.cigar_ops, n_ops, np.uint32))

    def align_batch_host_raw(self, c_batch: sdp_batch) -> sdp_result:
        """sdp_align_batch_host on a prepared sdp_batch of host pointers; result stays in the ctx's pinned memory."""
        res = sdp_result()
        self._check(self._lib.sdp_align_batch_host(self._h, ctypes.byref(c_batch), ctypes.byref(res)))
        return res
