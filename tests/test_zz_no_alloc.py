"""sdp_best_per_read_static: the per-read choice for callers that cannot allocate GPU memory.

Some users of libsdp run inside a program that claimed the whole card for its own buffers at start-up, or that keeps
other streams busy and cannot afford the device-wide stall of cudaMalloc / cudaFree. For them the library has one
entry point that allocates nothing: the caller brings inputs and outputs, and the per-read keys live in a fixed 8 MiB
array inside libsdp.so (limit: SDP_STATIC_MAX_READS = 2**20 reads per call). These tests hold it to the existing
path, sdp_best_per_read, bit for bit (all outputs are integers), on two calls in a row that share that array.

The file sorts after every other test file on purpose: pytest -x stops at the first failure, and a failure here must
not hide the parity tests. It passes alone in a fresh process and after the rest of the suite."""
import numpy as np
import pytest

from paper_1302_5507_b200 import workloads as W

FIELDS = ("best_pair", "best_score", "second_score", "n_candidates")


def _static_choice(S, torch, db, res, n_reads, out):
    """One call of the no-allocation entry point into the first n_reads entries of the caller's four arrays."""
    S.best_per_read_static(db.tensors["pairs"], res.score, db.n_pairs, n_reads, out["best_pair"], out["best_score"],
                           out["second_score"], out["n_candidates"], device=0)
    torch.cuda.synchronize()
    return {k: out[k][:n_reads].cpu().numpy() for k in FIELDS}


def _same(exp, got, what):
    for k in FIELDS:
        # best_pair / n_candidates are unsigned on the library side and int32 tensors here: compare the bit patterns
        a, b = exp[k].astype(np.int64) & 0xFFFFFFFF, got[k].astype(np.int64) & 0xFFFFFFFF
        assert np.array_equal(a, b), f"{what}: {k} differs from sdp_best_per_read at reads {np.flatnonzero(a != b)[:8]}"


@pytest.mark.gpu
def test_static_choice_equals_context_path_on_two_calls_in_a_row():
    import torch
    import paper_1302_5507_b200 as S
    big = W.make_step3(700, max_candidates=30, ref_bases=1_000_000)
    small = W.make_step3(260, max_candidates=12, ref_bases=400_000, seed=77)
    # everything the two calls write into exists before the first of them
    out = {k: torch.empty(len(big.read_len), dtype=torch.int32, device="cuda:0") for k in FIELDS}
    with S.Context(device=0) as ctx:
        ctx.set_score_only(True)                       # the choice needs scores only
        db = ctx.upload(big)
        res = ctx.align_batch(db)
        exp = ctx.best_per_read(db, res)
        got = _static_choice(S, torch, db, res, len(big.read_len), out)
        _same(exp, got, "first call")
        assert (got["n_candidates"] > 0).all() and got["n_candidates"].sum() == big.n_pairs

        # second call, fewer reads, other scores: the fixed array still holds the first call's keys, which would
        # outrank many of the new ones if the entry point did not clear them
        db2 = ctx.upload(small)
        res2 = ctx.align_batch(db2)
        exp2 = ctx.best_per_read(db2, res2)
        for k in FIELDS:
            out[k].fill_(-7)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info(0)[0]
        got2 = _static_choice(S, torch, db2, res2, len(small.read_len), out)
        free_after = torch.cuda.mem_get_info(0)[0]
        _same(exp2, got2, "second call")
        assert free_after == free_before, "the no-allocation entry point changed the device's free memory"
        # entries past n_reads belong to the caller and stay as they were
        assert all(bool((out[k][len(small.read_len):] == -7).all()) for k in FIELDS)


@pytest.mark.gpu
def test_static_choice_refuses_more_reads_than_its_fixed_array_holds():
    import torch
    import paper_1302_5507_b200 as S
    from paper_1302_5507_b200 import binding
    one = torch.zeros(2, dtype=torch.int32, device="cuda:0")
    with pytest.raises(S.SdpError) as e:
        S.best_per_read_static(one, one, 1, binding.SDP_STATIC_MAX_READS + 1, one, one, one, one, device=0)
    assert e.value.code == binding.SDP_ERANGE and "SDP_STATIC_MAX_READS" in str(e.value)
    torch.cuda.synchronize()
    assert int(one.sum()) == 0                          # refused before touching anything
