"""mstar_paged_attn_decode_static: the decode call whose scratch is a static device array inside the library (no
allocation on the call path; include/mstar_attn.h).  Collected last on purpose (the suite runs with pytest -x).
The new entry point against the existing path (mstar_paged_attn_decode with a caller-owned workspace) on calls made
back to back with different geometries -- the array keeps the previous call's contents, nothing is cleared in
between -- within the gates of every other parity test (tests/util.py: max-abs 2e-2, row-rel 1e-2), and bit for bit,
since the two run the same kernels; the first batch also against the fp64 oracle.  Independent of test order: it
passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_12688_b200 as mstar
import workloads as W
from tests.util import check_parity, compact_pool_after_append, decode_q

pytestmark = pytest.mark.gpu


def _batch(seed, lens, Hq, Hkv, D, p):
    pages = sum((l + p - 1) // p for l in lens)
    return W.make_batch(np.random.default_rng(seed), "no_alloc", lens, [min(1, l) for l in lens], Hq, Hkv, D, p,
                        2 * pages + 3)


def _existing(db, parts):
    out, lse = db.decode(num_partitions=parts)
    return out, lse


def _static(db, parts):
    b = db.b
    dev = db.q_decode.device
    out = torch.full((b.num_seqs, b.num_q_heads, b.head_dim), float("nan"), dtype=torch.bfloat16, device=dev)
    lse = torch.full((b.num_seqs, b.num_q_heads), float("nan"), dtype=torch.float32, device=dev)
    mstar.paged_attn_decode_static(out, db.q_decode, db.pool, db.block_table, db.seq_lens, b.max_seq_len,
                                   float(b.scale), num_partitions=parts, lse_out=lse)
    return out, lse


def _same(got, want, what):
    from tests.gpu_util import f64_of
    (o, l), (wo, wl) = got, want
    check_parity(f64_of(o), f64_of(wo), what)
    gl, wl64 = f64_of(l), f64_of(wl)
    assert np.array_equal(np.isneginf(gl), np.isneginf(wl64)), what
    fin = np.isfinite(wl64)
    assert np.abs(gl[fin] - wl64[fin]).max(initial=0.0) < 2e-3, what
    # same kernels, same launches: identical bits
    assert torch.equal(o.view(torch.int16), wo.view(torch.int16)), what + ": outputs differ in bits"
    assert torch.equal(l.view(torch.int32), wl.view(torch.int32)), what + ": LSEs differ in bits"


def test_decode_static_equals_existing_path_on_calls_in_a_row():
    from tests.gpu_util import DeviceBatch, f64_of
    # A: ragged, balanced tile ranges (streams cut by CTA ranges, empty and one-token sequences), D 128 / page 16
    a = _batch(11, [0, 1, 17, 64, 65, 700, 3000, 5000, 129, 2049, 4096, 33], 28, 4, 128, 16)
    # B: another geometry and the fixed-partition mode (3 partitions, the last ones empty for short rows), D 64 / page 32
    b = _batch(12, [100, 1, 333, 64, 2500, 900, 31], 8, 2, 64, 32)
    da, dbb = DeviceBatch(a), DeviceBatch(b)
    da.append()
    dbb.append()
    # the new entry point, calls in a row on one stream, nothing cleared in between
    sa1 = _static(da, 0)
    sb = _static(dbb, 3)
    sa2 = _static(da, 0)
    sa16 = _static(da, 16)
    torch.cuda.synchronize()
    _same(sa1, _existing(da, 0), "static A (first call)")
    _same(sb, _existing(dbb, 3), "static B (second call, other geometry)")
    _same(sa2, _existing(da, 0), "static A again (after B left its partials in the array)")
    _same(sa16, _existing(da, 16), "static A, 16 fixed partitions")
    # and against the definition
    k, v = compact_pool_after_append(a)
    want, want_lse = oracle.paged_decode(decode_q(a), k, v, a.compact_block_table, a.seq_lens, a.scale)
    check_parity(f64_of(sa2[0]), want, "static A vs oracle")
    got_lse = f64_of(sa2[1])
    fin = np.isfinite(want_lse)
    assert np.array_equal(np.isneginf(got_lse), np.isneginf(want_lse))
    assert np.abs(got_lse[fin] - want_lse[fin]).max(initial=0.0) < 2e-3


def test_decode_static_serving_shape_then_small_call():
    """The BAGEL-like CFG-pair batch (configs[1], 29.8 MB of partial slots) fills most of the array; a small call
    right behind it sees its leftovers."""
    from tests.gpu_util import DeviceBatch
    b2 = W.config2_bagel_cfg_decode()
    d2 = DeviceBatch(b2)
    d2.append()
    small = _batch(13, [5, 2000, 64, 0, 1500], 16, 2, 128, 16)
    ds = DeviceBatch(small)
    ds.append()
    s2 = _static(d2, 0)
    ss = _static(ds, 0)
    torch.cuda.synchronize()
    _same(s2, _existing(d2, 0), "static configs[1]")
    _same(ss, _existing(ds, 0), "static small call behind configs[1]")


def test_decode_static_rejects_geometries_beyond_the_array():
    """64 sequences x 32 heads x 64 partitions x (128 + 2) floats = 68 MB > 48 MiB: refused, nothing launched."""
    from tests.gpu_util import DeviceBatch
    assert mstar.MSTAR_DECODE_STATIC_WORKSPACE_BYTES == 48 << 20
    b = _batch(14, [40] * 64, 32, 4, 128, 16)
    d = DeviceBatch(b)
    d.append()
    need = mstar.decode_workspace_bytes(64, 32, 128, 64)
    assert need > mstar.MSTAR_DECODE_STATIC_WORKSPACE_BYTES
    out = torch.full((64, 32, 128), 7.0, dtype=torch.bfloat16, device="cuda")
    lib = mstar.load_library()
    import ctypes
    rc = lib.mstar_paged_attn_decode_static(out.data_ptr(), None, d.q_decode.data_ptr(), ctypes.byref(d.pool.c),
                                            d.block_table.data_ptr(), int(d.block_table.stride(0)),
                                            d.seq_lens.data_ptr(), 64, 32, 8192, float(b.scale), 64, 0, None)
    assert rc == -3 and "workspace" in mstar.status_string(rc).lower()
    assert mstar.last_launch_count() == 0
    with pytest.raises(mstar.MstarError, match="static array"):
        mstar.paged_attn_decode_static(out, d.q_decode, d.pool, d.block_table, d.seq_lens, 8192, float(b.scale),
                                       num_partitions=64)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())          # untouched
    # the same rows with a number of partitions that fits are served
    got = _static(d, 4)
    torch.cuda.synchronize()
    _same(got, _existing(d, 4), "static, 4 partitions")
