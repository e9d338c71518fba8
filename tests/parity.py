"""Element-by-element comparison of the CUDA path (through the C ABI) with the CPU oracle."""
import os

import numpy as np

import oracle
from oracle import OracleScoring
from paper_1302_5507_b200 import workloads as W

FIELDS = ["score", "ref_end", "ref_start", "read_start", "read_end", "n_match", "n_cols", "passed", "cigar_len",
          "cigar_off"]


def run_oracle(batch, sc: OracleScoring, threads=None, local=False):
    threads = threads or os.cpu_count() or 1
    return oracle.align_batch(batch.reads_packed, batch.read_off, batch.read_len, batch.wins_packed, batch.win_off,
                              batch.win_len, batch.pairs, sc, read_nmask=batch.read_nmask,
                              win_nmask=batch.win_nmask, threads=threads, local=local)


def describe(batch, p, exp, got):
    ri, wi = (int(x) for x in batch.pairs[p])
    n, m = int(batch.read_len[ri]), int(batch.win_len[wi])
    R = W.unpack(batch.reads_packed, int(batch.read_off[ri]), n, batch.read_nmask)
    T = W.unpack(batch.wins_packed, int(batch.win_off[wi]), m, batch.win_nmask)
    lines = [f"pair {p}: read {ri} (n={n}) window {wi} (m={m})", f"  R={R}", f"  T={T}"]
    for name, r in (("oracle", exp), ("cuda", got)):
        lines.append(f"  {name}: score={r.score[p]} ref=[{r.ref_start[p]},{r.ref_end[p]}] n_match={r.n_match[p]} "
                     f"n_cols={r.n_cols[p]} pass={r.passed[p]} cigar={r.cigar(p)}")
    return "\n".join(lines)


def assert_equal(batch, exp, got, what=""):
    """Bit-exact on every output array (reading R14: there is exactly one right answer)."""
    for f in FIELDS:
        a, b = getattr(exp, f), getattr(got, f)
        assert a.shape == b.shape, (what, f, a.shape, b.shape)
        bad = np.nonzero(a.astype(np.int64) != b.astype(np.int64))[0]
        if len(bad):
            raise AssertionError(f"{what}: {len(bad)} of {len(a)} pairs differ in '{f}'; first:\n"
                                 + describe(batch, int(bad[0]), exp, got))
    assert exp.cigar_ops.shape == got.cigar_ops.shape, (what, "cigar_ops", exp.cigar_ops.shape, got.cigar_ops.shape)
    bad = np.nonzero(exp.cigar_ops != got.cigar_ops)[0]
    if len(bad):
        p = int(np.searchsorted(exp.cigar_off, bad[0], side="right") - 1)
        raise AssertionError(f"{what}: cigar_ops differ; first:\n" + describe(batch, p, exp, got))


def check_batch(ctx, batch, sc: OracleScoring, what="", host_path=True, local=False):
    """`local` must match the mode the ctx was put in (Context.set_mode)."""
    exp = run_oracle(batch, sc, local=local)
    db = ctx.upload(batch)
    got = ctx.fetch(ctx.align_batch(db))
    assert_equal(batch, exp, got, what + " [device path]")
    if host_path:
        got_h = ctx.align_batch_host(batch)
        assert_equal(batch, exp, got_h, what + " [host path]")
    return exp, got
