"""GPU parity of the quantised (fp8 E4M3) K/V pool against oracle/fp8.py: the quantising
append bit-exact over the whole pool, decode within the gates of DESIGN.md R11 on the same codes.  Needs a B200."""
import numpy as np
import pytest
import torch

import paper_2606_12688_b200 as mstar
import workloads as W
from oracle import fp8 as ofp8
from tests.gpu_util import DeviceBatchFp8, bf16_tensor, f64_of
from tests.util import check_parity, decode_q

pytestmark = pytest.mark.gpu


def small_batch(seed, lens, Hq=8, Hkv=2, p=16, pool=None, **kw):
    rng = np.random.default_rng(seed)
    q_lens = [min(1, l) for l in lens]
    pages = sum((l + p - 1) // p for l in lens)
    return W.make_batch(rng, "t8", lens, q_lens, Hq, Hkv, 128, p, pool or max(2 * pages, 4), **kw)


def oracle_pool(b, k_scale, v_scale):
    """The oracle's quantised compact store after the step: store rows, then the new rows, through APPEND_FP8."""
    U, Hkv, p, D = b.k_store.shape
    k8 = np.full((U, Hkv, p, D), 0x7F, dtype=np.uint8)
    v8 = np.full((U, Hkv, p, D), 0x7F, dtype=np.uint8)
    ks, vs = k_scale[b.used_pages], v_scale[b.used_pages]  # scales of the compact store's pages
    rows_k = b.k_store.transpose(0, 2, 1, 3).reshape(-1, Hkv, D)
    rows_v = b.v_store.transpose(0, 2, 1, 3).reshape(-1, Hkv, D)
    ofp8.kv_append_fp8(k8, v8, ks, vs, rows_k, rows_v, np.arange(U * p, dtype=np.int64))
    ofp8.kv_append_fp8(k8, v8, ks, vs, b.k_new, b.v_new, b.compact_slot_mapping)
    return k8, v8, ks, vs


def run_case(b, parts_list=(0,), layout="HND", seed=1, scale_range=(0.006, 0.02)):
    k_scale, v_scale = W.fp8_page_scales(seed, b.num_pages, b.num_kv_heads, lo=scale_range[0], hi=scale_range[1])
    db = DeviceBatchFp8(b, k_scale, v_scale, layout=layout)
    db.quantise_store()
    db.append()
    k8, v8, ks, vs = oracle_pool(b, k_scale, v_scale)
    gk, gv = db.store_codes()
    assert np.array_equal(gk, k8) and np.array_equal(gv, v8), "quantised codes differ from the oracle"
    # pages no sequence uses keep their poison
    unused = np.setdiff1d(np.arange(b.num_pages), b.used_pages)
    if unused.size:
        idx = torch.from_numpy(unused[:64]).to(db.k_pool.device)
        assert bool((db.k_pool[idx] == 0x7F).all()) and bool((db.v_pool[idx] == 0x7F).all())
    want, want_lse = ofp8.paged_decode_fp8(decode_q(b), k8, v8, ks, vs, b.compact_block_table, b.seq_lens, b.scale)
    stats = {}
    for parts in parts_list:
        out, lse = db.decode(num_partitions=parts)
        stats[parts] = check_parity(f64_of(out), want, "%s fp8 parts=%d" % (b.name, parts))
        got_lse = f64_of(lse)
        fin = np.isfinite(want_lse)
        assert np.array_equal(np.isneginf(got_lse), np.isneginf(want_lse))
        assert np.abs(got_lse[fin] - want_lse[fin]).max(initial=0.0) < 2e-3
    out32, _ = db.decode(num_partitions=parts_list[0], out_dtype=torch.float32)
    _, r = check_parity(f64_of(out32), want, "%s fp8 f32" % b.name)
    assert r <= 6e-3
    return stats


@pytest.mark.parametrize("layout", ["HND", "NHD"])
def test_append_fp8_bit_exact_with_skips_and_special_values(layout):
    b = small_batch(31, [0, 1, 15, 16, 17, 100, 257], Hq=8, Hkv=2, p=16)
    # special inputs in the new rows: huge, tiny, zero, negative zero, NaN, inf
    b.k_new[0, 0, :6] = W.bf16_bits_from_f32(np.array([1e30, -1e30, 1e-30, 0.0, -0.0, np.inf], dtype=np.float32))
    b.v_new[0, 0, 0] = W.BF16_NAN
    b.slot_mapping[2] = -1
    b.compact_slot_mapping[2] = -1
    k_scale, v_scale = W.fp8_page_scales(2, b.num_pages, b.num_kv_heads)
    db = DeviceBatchFp8(b, k_scale, v_scale, layout=layout)
    db.quantise_store()
    db.append()
    k8, v8, _, _ = oracle_pool(b, k_scale, v_scale)
    gk, gv = db.store_codes()
    assert np.array_equal(gk, k8) and np.array_equal(gv, v8)


@pytest.mark.parametrize("p", [16, 32])
@pytest.mark.parametrize("G", [1, 4, 7, 8, 16])
def test_decode_fp8_edge_lengths(p, G):
    lens = [0, 1, p - 1, p, p + 1, 2 * p - 1, 63, 64, 65, 127, 128, 129, 191, 257, 300]
    b = small_batch(300 + G, lens, Hq=G * 2, Hkv=2, p=p, table_width=40)
    run_case(b, parts_list=(0, 1, 3, 9))


@pytest.mark.parametrize("Hkv,G", [(1, 8), (8, 4), (1, 12)])
def test_decode_fp8_kv_head_counts(Hkv, G):
    b = small_batch(380 + Hkv + G, [700, 1, 65, 300, 129], Hq=Hkv * G, Hkv=Hkv, p=32)
    run_case(b, parts_list=(0, 3))


def test_decode_fp8_many_sequences_nhd_and_long_stream():
    rng = np.random.default_rng(17)
    lens = rng.integers(1, 500, 149).tolist()
    lens[70] = 5000
    b = small_batch(310, lens, Hq=8, Hkv=4, p=16)
    run_case(b, parts_list=(0, 4), layout="NHD")


@pytest.mark.parametrize("p,G", [(16, 7), (32, 4), (16, 1)])
def test_decode_fp8_long_sequences_take_the_12_warp_kernel(p, G):
    """max_seq_len > 8192 and G <= 8 select 12 consumer warps on 192-token stages: lengths around the stage and
    partition boundaries of that geometry, next to one long stream."""
    lens = [9000, 0, 1, 191, 192, 193, 383, 385, 16 * 192 + 5, 2111, 2113]
    b = small_batch(360 + G, lens, Hq=G * 2, Hkv=2, p=p, table_width=9000 // p + 8)
    run_case(b, parts_list=(0, 1, 5, 16))


def test_decode_fp8_len1_is_the_dequantised_v_row():
    b = small_batch(320, [1, 1, 1], Hq=8, Hkv=2, p=16)
    k_scale, v_scale = W.fp8_page_scales(3, b.num_pages, b.num_kv_heads)
    db = DeviceBatchFp8(b, k_scale, v_scale)
    db.append()
    out32, _ = db.decode(num_partitions=1, out_dtype=torch.float32)
    k8, v8, ks, vs = oracle_pool(b, k_scale, v_scale)
    t = ofp8.e4m3_decode_table()
    got = f64_of(out32)
    for s in range(3):
        pg = int(b.compact_block_table[s, 0])
        for h in range(8):
            g = h // 4
            # p = 1, l = 1: the row is the code values times v_scale.  The kernel folds v_scale into P as a bf16
            # operand and, in items of a single stage, feeds the residual of that rounding through a second MMA: what
            # is left is 2^-16 relative (before that residual pass the row was codes * bf16(v_scale), 2^-8 relative)
            want = t[v8[pg, g, 0]] * float(vs[pg, g])
            assert np.all(np.abs(got[s, h] - want) <= np.abs(want) * 2.0 ** -15)


def test_decode_fp8_short_rows_found_by_the_soak_run():
    """The example the property tests found at 20 x their examples (MSTAR_SOAK=20): rows of one token whose |v| is
    3.4, where the rounding of p * v_scale to a bf16 operand and the output rounding added up to 2.03e-2.  Single-stage
    items now carry the residual of that rounding through a second MMA."""
    from tests.test_properties import decode_batch
    seed, p, G, L = 195, 32, 4, [1, 257, 1, 33, 257]
    b = decode_batch(seed, (p, 128, G, 2), L)
    ks, vs = W.fp8_page_scales(seed % 97, b.num_pages, b.num_kv_heads)
    db = DeviceBatchFp8(b, ks, vs)
    db.quantise_store()
    db.append()
    k8, v8, cks, cvs = oracle_pool(b, ks, vs)
    want, _ = ofp8.paged_decode_fp8(decode_q(b), k8, v8, cks, cvs, b.compact_block_table, b.seq_lens, b.scale)
    for parts in (0, 1, 3):
        out, _ = db.decode(num_partitions=parts)
        a, _ = check_parity(f64_of(out), want, "soak example parts=%d" % parts)
        assert a <= 1.6e-2     # |out| < 4: the output's own rounding is 7.8e-3, the rest is the arithmetic's


def test_decode_fp8_subnormal_codes_are_exact():
    """Scales so large that almost every code is an E4M3 subnormal (|x / scale| < 2^-6): the kernel's byte -> bf16
    conversion maps them to bf16 subnormals, which must survive the tensor core (a flush would zero K and V)."""
    b = small_batch(340, [1, 40, 130, 700], Hq=8, Hkv=2, p=16)
    k_scale = np.full((b.num_pages, b.num_kv_heads), 96.0, dtype=np.float32)
    v_scale = np.full((b.num_pages, b.num_kv_heads), 160.0, dtype=np.float32)
    db = DeviceBatchFp8(b, k_scale, v_scale)
    db.quantise_store()
    db.append()
    k8, v8, ks, vs = oracle_pool(b, k_scale, v_scale)
    used = k8[b.compact_block_table[3, :40]]
    assert ((used & 0x78) == 0).mean() > 0.7 and (used & 0x7F).max() > 0  # mostly subnormal codes, not all zero
    want, _ = ofp8.paged_decode_fp8(decode_q(b), k8, v8, ks, vs, b.compact_block_table, b.seq_lens, b.scale)
    assert np.abs(want).max() > 0.5
    for parts in (0, 1, 4):
        out, _ = db.decode(num_partitions=parts)
        check_parity(f64_of(out), want, "subnormal codes parts=%d" % parts)


def test_fp8_deterministic_graph_capturable_and_page_permutation_invariant():
    b = small_batch(350, [500, 123, 64, 1], Hq=14, Hkv=2, p=16, pool=80)
    k_scale, v_scale = W.fp8_page_scales(5, b.num_pages, b.num_kv_heads)
    db = DeviceBatchFp8(b, k_scale, v_scale)
    db.quantise_store()
    S, Hq, D = 4, 14, 128
    out = torch.zeros((S, Hq, D), dtype=torch.bfloat16, device="cuda")
    ws = torch.empty(mstar.decode_workspace_bytes(S, Hq, D, 4), dtype=torch.uint8, device="cuda")

    def step(bt=None):
        db.append()
        mstar.paged_attn_decode_fp8(out, db.q_decode, db.pool, db.block_table if bt is None else bt, db.seq_lens,
                                    500, float(b.scale), num_partitions=4, workspace=ws)

    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        step()
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    first = out.clone()
    codes_first = db.store_codes()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        step()
    out.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(first.view(torch.int16), out.view(torch.int16))
    assert all(np.array_equal(a, c) for a, c in zip(codes_first, db.store_codes()))
    # relabel the physical pages of sequence 0 (codes and scales move with them): bit-identical output
    used = np.zeros(b.num_pages, dtype=bool)
    used[b.used_pages] = True
    free = np.flatnonzero(~used)
    bt2 = db.block_table.clone()
    npg = (500 + 15) // 16
    for i in range(npg):
        src, dst = int(bt2[0, i]), int(free[i])
        db.k_pool[dst] = db.k_pool[src]
        db.v_pool[dst] = db.v_pool[src]
        db.k_scale[dst] = db.k_scale[src]
        db.v_scale[dst] = db.v_scale[src]
        bt2[0, i] = dst
    out.zero_()
    mstar.paged_attn_decode_fp8(out, db.q_decode, db.pool, bt2, db.seq_lens, 500, float(b.scale), num_partitions=4,
                                workspace=ws)
    torch.cuda.synchronize()
    assert torch.equal(first.view(torch.int16), out.view(torch.int16))


def test_decode_fp8_config2_bagel_cfg_pairs():
    b = W.config2_bagel_cfg_decode()
    stats = run_case(b, parts_list=(0,))
    print("config 2 fp8", stats)


def test_fp8_page_moves_through_the_bit_pool_view():
    """mstar_kv_copy_pages / mstar_kv_gather on the quantised pool described as a bf16 pool of head_dim 64: moved pages
    (codes by the kernel, scale rows by the caller) decode bit-identically; gathered rows equal the oracle's codes."""
    b = small_batch(390, [300, 77, 1], Hq=8, Hkv=2, p=16, pool=96)
    k_scale, v_scale = W.fp8_page_scales(6, b.num_pages, b.num_kv_heads)
    db = DeviceBatchFp8(b, k_scale, v_scale)
    db.quantise_store()
    db.append()
    out0, _ = db.decode(num_partitions=2)
    bits = db.pool.as_bit_pool()
    used = np.zeros(b.num_pages, dtype=bool)
    used[b.used_pages] = True
    free = np.flatnonzero(~used)[:len(b.used_pages)].astype(np.int64)
    src = torch.from_numpy(b.used_pages.astype(np.int64)).cuda()
    dst = torch.from_numpy(free).cuda()
    mstar.kv_copy_pages(bits, bits, dst, src)
    db.k_scale[dst] = db.k_scale[src]
    db.v_scale[dst] = db.v_scale[src]
    remap = np.full(b.num_pages, -1, dtype=np.int32)
    remap[b.used_pages] = free
    bt2 = np.where(b.block_table >= 0, remap[np.maximum(b.block_table, 0)], -1).astype(np.int32)
    db.block_table = torch.from_numpy(bt2).cuda()
    db.k_pool[src] = 0x7F  # the old pages are poison now
    db.v_pool[src] = 0x7F
    out1, _ = db.decode(num_partitions=2)
    assert torch.equal(out0.view(torch.int16), out1.view(torch.int16))
    # gather the codes of every sequence to contiguous rows
    cu = np.zeros(b.num_seqs + 1, dtype=np.int32)
    cu[1:] = np.cumsum(b.seq_lens)
    kg = torch.zeros((int(cu[-1]), b.num_kv_heads, 64), dtype=torch.bfloat16, device="cuda")
    vg = torch.zeros_like(kg)
    mstar.kv_gather(kg, vg, bits, db.block_table, db.seq_lens, torch.from_numpy(cu).cuda())
    k8, v8, _, _ = oracle_pool(b, k_scale, v_scale)
    gk = kg.view(torch.uint8).cpu().numpy()
    for s in range(b.num_seqs):
        for j in range(int(b.seq_lens[s])):
            pg = int(b.compact_block_table[s, j // 16])
            assert np.array_equal(gk[cu[s] + j], k8[pg, :, j % 16, :])


def test_fp8_error_codes():
    b = small_batch(330, [5], Hq=8, Hkv=2, p=16)
    dev = "cuda"
    k = torch.zeros((4, 2, 16, 64), dtype=torch.uint8, device=dev)
    sc = torch.ones((4, 2), dtype=torch.float32, device=dev)
    pool64 = mstar.KVPoolFp8(k, k.clone(), sc, sc)
    q = torch.zeros((1, 8, 64), dtype=torch.bfloat16, device=dev)
    out = torch.zeros_like(q)
    bt = torch.zeros((1, 1), dtype=torch.int32, device=dev)
    sl = torch.ones(1, dtype=torch.int32, device=dev)
    with pytest.raises(mstar.MstarError, match="UNSUPPORTED"):
        mstar.paged_attn_decode_fp8(out, q, pool64, bt, sl, 1, 0.125, num_partitions=1)


# ----------------------------------------------------------------------------- prefill / flow step over the fp8 pool

def prefill_batch(seed, lens, q_lens, Hq=8, Hkv=2, p=16, **kw):
    rng = np.random.default_rng(seed)
    pages = sum((l + p - 1) // p for l in lens)
    return W.make_batch(rng, "p8", lens, q_lens, Hq, Hkv, 128, p, max(2 * pages, 4), **kw)


def run_prefill_case(b, causal=True, layout="HND", seed=2, rows=None, check_f32=True):
    """mstar_kv_append_fp8 (store + new rows; codes bit-exact against APPEND_FP8) then
    mstar_paged_attn_prefill_fp8 against PREFILL_FP8 on the oracle's codes (gates R11)."""
    k_scale, v_scale = W.fp8_page_scales(seed, b.num_pages, b.num_kv_heads)
    db = DeviceBatchFp8(b, k_scale, v_scale, layout=layout)
    db.quantise_store()
    db.append()
    k8, v8, ks, vs = oracle_pool(b, k_scale, v_scale)
    gk, gv = db.store_codes()
    assert np.array_equal(gk, k8) and np.array_equal(gv, v8), "quantised codes differ from the oracle"
    want, want_lse = ofp8.paged_prefill_fp8(b.q, b.cu_seqlens_q, k8, v8, ks, vs, b.compact_block_table, b.seq_lens,
                                            b.scale, causal=causal, rows=rows)
    sel = slice(None) if rows is None else np.asarray(rows)
    out, lse = db.prefill(causal=causal)
    stats = check_parity(f64_of(out)[sel], want, "%s fp8 prefill causal=%d" % (b.name, causal))
    assert np.abs(f64_of(lse)[sel] - want_lse).max(initial=0.0) < 2e-3
    if check_f32:
        out32, _ = db.prefill(causal=causal, out_dtype=torch.float32)
        _, r = check_parity(f64_of(out32)[sel], want, "%s fp8 prefill f32" % b.name)
        assert r <= 6e-3
    return stats


@pytest.mark.parametrize("p", [16, 32])
@pytest.mark.parametrize("G", [1, 4, 7, 8, 12])
@pytest.mark.parametrize("causal", [True, False])
def test_prefill_fp8_ragged_small(p, G, causal):
    """Ragged batch with cached prefixes: rows per sequence 1 .. 200, prefixes 0 .. 300, an empty sequence."""
    lens = [200 + 40, 64, 33 + 300, 1, 0, 129 + 16]
    q_lens = [200, 64, 33, 1, 0, 129]
    b = prefill_batch(40 + G, lens, q_lens, Hq=G * 2, Hkv=2, p=p)
    run_prefill_case(b, causal=causal)


def test_prefill_fp8_new_tokens_times_prefix_matrix_and_nhd_layout():
    ns, Ps = [1, 2, 127, 128, 129], [0, 1, 15, 16, 255, 256]
    lens, q_lens = [], []
    for n in ns:
        for P in Ps:
            lens.append(n + P)
            q_lens.append(n)
    b = prefill_batch(77, lens, q_lens, Hq=8, Hkv=2, p=16)
    run_prefill_case(b, causal=True, layout="NHD", check_f32=False)


def test_prefill_fp8_kv_head_counts():
    for Hkv, G in ((1, 8), (8, 4)):
        b = prefill_batch(90 + Hkv, [150, 70, 260], [100, 70, 4], Hq=Hkv * G, Hkv=Hkv, p=16)
        run_prefill_case(b, check_f32=False)


def test_prefill_fp8_long_block_over_prefix_and_flow_step_sampled_rows():
    """1024 new tokens over a 700-token prefix (causal) and a bidirectional 1024-token block over two label contexts
    that share pages (the flow step, causal = 0), compared on sampled rows."""
    b = prefill_batch(5, [1724, 1024 + 1], [1024, 1024], Hq=28, Hkv=4, p=16)
    rows = np.unique(np.concatenate([np.random.default_rng(0).integers(0, 2048, 40), [0, 1023, 1024, 2047]]))
    print("fp8 prefill causal", run_prefill_case(b, causal=True, rows=rows, check_f32=False))
    bf = prefill_batch(6, [1024 + 64, 1024 + 64], [1024, 1024], Hq=28, Hkv=4, p=16, share_with=[-1, 0],
                       shared_tokens=64)
    print("fp8 flow step", run_prefill_case(bf, causal=False, rows=rows, check_f32=False))


def test_prefill_fp8_deterministic_graph_capturable_and_error_codes():
    b = prefill_batch(8, [300, 90], [128, 90], Hq=8, Hkv=2, p=16)
    k_scale, v_scale = W.fp8_page_scales(3, b.num_pages, b.num_kv_heads)
    db = DeviceBatchFp8(b, k_scale, v_scale)
    db.quantise_store()
    db.append()
    o1, _ = db.prefill()
    o2, _ = db.prefill()
    assert torch.equal(o1.view(torch.int16), o2.view(torch.int16))
    T, Hq, D = b.total_q, b.num_q_heads, b.head_dim
    q = bf16_tensor(b.q)
    cu = torch.from_numpy(b.cu_seqlens_q).cuda()
    ws = torch.empty(mstar.prefill_fp8_workspace_bytes(b.num_seqs, T, Hq, b.num_kv_heads, b.page_size, b.max_seq_len),
                     dtype=torch.uint8, device="cuda")
    og = torch.empty_like(o1)
    call = lambda: mstar.paged_attn_prefill_fp8(og, q, cu, db.pool, db.block_table, db.seq_lens, b.max_q_len,
                                                b.max_seq_len, float(b.scale), workspace=ws)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        call()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            call()
    torch.cuda.synchronize()
    og.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(o1.view(torch.int16), og.view(torch.int16))
    with pytest.raises(mstar.MstarError, match="WORKSPACE_TOO_SMALL"):
        mstar.paged_attn_prefill_fp8(og, q, cu, db.pool, db.block_table, db.seq_lens, b.max_q_len, b.max_seq_len,
                                     float(b.scale), workspace=ws[:4096])
    with pytest.raises(mstar.MstarError, match="INVALID_ARG"):
        mstar.paged_attn_prefill_fp8(og, q, cu, db.pool, db.block_table, db.seq_lens, b.max_q_len, b.max_seq_len,
                                     -1.0, workspace=ws)


def test_prefill_fp8_config3_full_size_sampled_rows_every_sequence():
    """BASELINE configs[2] (8 x 1024 new tokens over cached prefixes, 28q / 4kv) on the quantised pool, the launch
    configuration bench.py times: sampled rows of every sequence incl. first and last rows."""
    b = W.config3_prefill()
    rng = np.random.default_rng(11)
    rows = np.unique(np.concatenate([rng.integers(0, b.total_q, 48), b.cu_seqlens_q[:-1], b.cu_seqlens_q[1:] - 1]))
    print("fp8 prefill config 3", run_prefill_case(b, causal=True, rows=rows, check_f32=False))


def test_decode_fp8_more_than_16_heads_per_kv_head():
    """Hq / Hkv = 32 on the quantised pool: two sub-groups of 16 heads over the same codes and scales."""
    b = small_batch(390, [1, 65, 700, 0, 129, 2300], Hq=32, Hkv=1, p=16)
    run_case(b, parts_list=(0, 1, 3))
