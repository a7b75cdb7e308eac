"""GPU parity: the CUDA path through the C ABI vs the fp64 oracle on the same seeded inputs.

Gates (R11, from BASELINE.json north_star): page scatter bit-exact; attention output
max-abs <= 2e-2 and per-row max-rel <= 1e-2 against the oracle.  All tests here need a B200.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_12688_b200 as mstar
import workloads as W
from tests.gpu_util import DeviceBatch, bf16_tensor, bits_of, f64_of
from tests.util import check_parity, compact_pool_after_append, decode_q, f64_from_bf16_bits

pytestmark = pytest.mark.gpu


def small_batch(seed, lens, q_lens=None, Hq=8, Hkv=2, D=64, p=16, pool=None, **kw):
    rng = np.random.default_rng(seed)
    q_lens = [min(1, l) for l in lens] if q_lens is None else q_lens
    pages = sum((l + p - 1) // p for l in lens)
    return W.make_batch(rng, "t", lens, q_lens, Hq, Hkv, D, p, pool or max(2 * pages, 4), **kw)


def oracle_decode(b):
    k, v = compact_pool_after_append(b)
    return oracle.paged_decode(decode_q(b), k, v, b.compact_block_table, b.seq_lens, b.scale)


def run_decode_case(b, parts_list=(0,), layout="HND", check_f32=True):
    db = DeviceBatch(b, layout=layout)
    db.append()
    want, want_lse = oracle_decode(b)
    stats = {}
    for parts in parts_list:
        out, lse = db.decode(num_partitions=parts)
        stats[parts] = check_parity(f64_of(out), want, "%s parts=%d" % (b.name, parts))
        got_lse = f64_of(lse)
        fin = np.isfinite(want_lse)
        assert np.array_equal(np.isneginf(got_lse), np.isneginf(want_lse))
        assert np.abs(got_lse[fin] - want_lse[fin]).max(initial=0.0) < 2e-3
        if check_f32:
            out32, _ = db.decode(num_partitions=parts, out_dtype=torch.float32)
            a, r = check_parity(f64_of(out32), want, "%s parts=%d f32" % (b.name, parts))
            assert r <= 6e-3  # without the bf16 output rounding the kernel error alone (bf16 P) must be smaller
    return stats


# ----------------------------------------------------------------------------- append

@pytest.mark.parametrize("layout", ["HND", "NHD"])
def test_append_bit_exact_whole_pool(layout):
    b = small_batch(101, [1, 17, 33, 100, 64], q_lens=[1, 5, 33, 40, 64], Hq=4, Hkv=2, D=128, p=16)
    db = DeviceBatch(b, layout=layout)
    db.append()
    torch.cuda.synchronize()
    k_ref, v_ref = b.full_pool()
    oracle.kv_append(k_ref, v_ref, b.k_new, b.v_new, b.slot_mapping)
    assert np.array_equal(bits_of(db.k_pool), k_ref)
    assert np.array_equal(bits_of(db.v_pool), v_ref)


def test_append_negative_slots_and_config3_scale():
    b = W.config3_prefill()
    db = DeviceBatch(b)
    slot = b.slot_mapping.copy()
    slot[::7] = -1
    db.slot_mapping = torch.from_numpy(slot).cuda()
    db.append()
    k_ref, v_ref = b.k_store.copy(), b.v_store.copy()
    cslot = b.compact_slot_mapping.copy()
    cslot[::7] = -1
    oracle.kv_append(k_ref, v_ref, b.k_new, b.v_new, cslot)
    kg, vg = db.store_rows_bits()
    assert np.array_equal(kg, k_ref) and np.array_equal(vg, v_ref)
    # pages no sequence references keep their poison
    unused = np.setdiff1d(np.arange(b.num_pages), b.used_pages)[:64]
    assert np.all(bits_of(db.k_pool[torch.from_numpy(unused).cuda()]) == 0x7FC0)


def test_build_slot_mapping_matches_generator():
    b = small_batch(102, [40, 17, 33, 5, 64], q_lens=[40, 1, 16, 5, 3], p=32)
    db = DeviceBatch(b)
    out = torch.full((b.total_q,), -5, dtype=torch.int64, device="cuda")
    mstar.build_slot_mapping(db.block_table, db.cu_seqlens_q, db.seq_lens, b.total_q, b.page_size, out)
    assert np.array_equal(out.cpu().numpy(), b.slot_mapping)


@pytest.mark.parametrize("layout", ["HND", "NHD"])
def test_gather_and_copy_pages_bit_exact(layout):
    """SURVEY 8(f) rank 4 page moves against the oracle: GATHER rows, COPY_PAGES into a second pool with the other
    layout and back into free pages of the same pool; whole pools compared bit for bit."""
    b = small_batch(150, [1, 17, 33, 100, 0, 257], q_lens=[1, 5, 33, 40, 0, 1], Hq=4, Hkv=2, D=128, p=16)
    db = DeviceBatch(b, layout=layout)
    db.append()
    k, v = b.full_pool()
    oracle.kv_append(k, v, b.k_new, b.v_new, b.slot_mapping)
    want_k, want_v, cu = oracle.kv_gather(k, v, b.block_table, b.seq_lens)
    k_out = torch.zeros((int(cu[-1]) + 3, 2, 128), dtype=torch.bfloat16, device="cuda")
    v_out = torch.zeros_like(k_out)
    mstar.kv_gather(k_out, v_out, db.pool, db.block_table, db.seq_lens, torch.from_numpy(cu).cuda())
    assert np.array_equal(bits_of(k_out)[:cu[-1]], want_k) and np.array_equal(bits_of(v_out)[:cu[-1]], want_v)
    assert not bits_of(k_out)[cu[-1]:].any()
    # pool -> other pool (other layout), sequence 5's pages to ids 0.., one skipped pair
    other = DeviceBatch(b, layout="NHD" if layout == "HND" else "HND")
    src = b.block_table[5, :17].astype(np.int64)
    dst = np.arange(17, dtype=np.int64) * 3 % b.num_pages
    src_s, dst_s = np.append(src, [2, -1]), np.append(dst, [-1, 2])
    k2, v2 = b.full_pool()
    oracle.kv_copy_pages(k2, v2, k, v, dst_s, src_s)
    mstar.kv_copy_pages(other.pool, db.pool, torch.from_numpy(dst_s).cuda(), torch.from_numpy(src_s).cuda())
    assert np.array_equal(bits_of(other.k_pool.contiguous()), k2)
    assert np.array_equal(bits_of(other.v_pool.contiguous()), v2)
    # same pool: to free pages, then attention through the relabelled block table is bit-identical
    used = set(b.used_pages.tolist())
    free = np.array([pg for pg in range(b.num_pages) if pg not in used][:17][::-1], dtype=np.int64)
    out0, _ = db.prefill()
    mstar.kv_copy_pages(db.pool, db.pool, torch.from_numpy(free).cuda(), torch.from_numpy(src).cuda())
    k3, v3 = k.copy(), v.copy()
    oracle.kv_copy_pages(k3, v3, k, v, free, src)
    assert np.array_equal(bits_of(db.k_pool.contiguous()), k3) and np.array_equal(bits_of(db.v_pool.contiguous()), v3)
    db.block_table[5, :17] = torch.from_numpy(free.astype(np.int32)).cuda()
    out1, _ = db.prefill()
    assert torch.equal(out0.view(torch.int16), out1.view(torch.int16))


# ----------------------------------------------------------------------------- decode

def test_decode_config1_tiny():
    run_decode_case(W.config1_tiny_decode(), parts_list=(0, 1, 2, 3, 16))


@pytest.mark.parametrize("D,p", [(64, 16), (64, 32), (128, 16), (128, 32)])
@pytest.mark.parametrize("G", [1, 2, 4, 7, 8, 16])
def test_decode_edge_lengths(D, p, G):
    """Lengths straddling page / stage (64) / partition boundaries, incl. L = 0 and L = 1."""
    lens = [0, 1, p - 1, p, p + 1, 2 * p - 1, 63, 64, 65, 127, 128, 129, 191, 257, 300]
    Hkv = 2
    b = small_batch(200 + G, lens, Hq=G * Hkv, Hkv=Hkv, D=D, p=p, table_width=40)
    run_decode_case(b, parts_list=(0, 1, 3, 9), check_f32=(G in (1, 7)))


@pytest.mark.parametrize("Hkv,G", [(1, 8), (1, 1), (8, 4), (8, 2)])
def test_decode_kv_head_counts(Hkv, G):
    """SURVEY 8(c) edge matrix: Hkv in {1, 8} (2 and 4 are what the other cases use)."""
    b = small_batch(260 + Hkv * 10 + G, [700, 1, 65, 300, 129], Hq=Hkv * G, Hkv=Hkv, D=128, p=32)
    run_decode_case(b, parts_list=(0, 3), check_f32=False)


def test_decode_many_sequences_and_nhd_layout():
    rng = np.random.default_rng(7)
    lens = rng.integers(1, 700, 300).tolist()
    b = small_batch(210, lens, Hq=8, Hkv=4, D=128, p=16)
    run_decode_case(b, parts_list=(0, 2), layout="NHD", check_f32=False)


@pytest.mark.parametrize("S", [1, 2, 3, 148, 149])
def test_decode_sequence_counts_and_balanced_cuts(S):
    """Batch sizes around the SM count; one long sequence among short ones makes the balanced mode
    (num_partitions = 0) cut a stream into many pieces (per = per_min) while other CTAs take whole streams."""
    rng = np.random.default_rng(230 + S)
    lens = rng.integers(1, 400, S).tolist()
    lens[S // 2] = 5000
    b = small_batch(230 + S, lens, Hq=14, Hkv=2, D=128, p=16)
    run_decode_case(b, parts_list=(0, 4), check_f32=False)


def test_decode_len1_bit_exact_and_unit_values():
    """Closed forms on the GPU: L = 1 => out = V row bit-for-bit; V == 1 => out == 1 exactly."""
    b = small_batch(220, [1, 1, 1, 200, 1000], Hq=8, Hkv=2, D=128, p=16)
    db = DeviceBatch(b)
    db.append()
    out, _ = db.decode(num_partitions=0)
    k, v = compact_pool_after_append(b)
    got = bits_of(out)
    for s in range(3):
        for h in range(8):
            assert np.array_equal(got[s, h], v[b.compact_block_table[s, 0], h // 4, 0])
    db.v_pool[~torch.isnan(db.v_pool)] = 1.0
    for parts in (0, 1, 5):
        out, _ = db.decode(num_partitions=parts)
        assert torch.all(out.float() == 1.0)


def test_decode_page_permutation_and_shared_prefix_bit_identical():
    lens = [300, 300, 77, 77]
    b = small_batch(230, lens, Hq=8, Hkv=2, D=128, p=16, share_with=[-1, 0, -1, 2], shared_tokens=64, pool=128)
    db = DeviceBatch(b)
    db.append()
    out1, _ = db.decode(num_partitions=3)
    # relabel physical pages: new id of old page i is perm[i]
    perm = torch.from_numpy(np.random.default_rng(5).permutation(b.num_pages)).cuda()
    k2, v2 = torch.empty_like(db.k_pool), torch.empty_like(db.v_pool)
    k2[perm], v2[perm] = db.k_pool, db.v_pool
    bt2 = torch.where(db.block_table >= 0, perm[db.block_table.clamp(min=0).long()].int(), db.block_table)
    out2 = torch.empty_like(out1)
    ws = torch.empty(mstar.decode_workspace_bytes(4, 8, 128, 3), dtype=torch.uint8, device="cuda")
    mstar.paged_attn_decode(out2, db.q_decode, mstar.KVPool(k2, v2), bt2.contiguous(), db.seq_lens, 300, float(b.scale),
                            num_partitions=3, workspace=ws)
    assert torch.equal(out1.view(torch.int16), out2.view(torch.int16))
    # duplicated prefix: sequence 1 gets private copies of the shared pages
    free = np.setdiff1d(np.arange(b.num_pages), b.used_pages)
    bt3 = db.block_table.clone()
    for i in range(4):
        db.k_pool[free[i]] = db.k_pool[bt3[1, i].item()]
        db.v_pool[free[i]] = db.v_pool[bt3[1, i].item()]
        bt3[1, i] = int(free[i])
    out3 = torch.empty_like(out1)
    mstar.paged_attn_decode(out3, db.q_decode, db.pool, bt3, db.seq_lens, 300, float(b.scale), num_partitions=3,
                            workspace=ws)
    assert torch.equal(out1.view(torch.int16), out3.view(torch.int16))


def test_decode_deterministic_and_graph_capturable():
    b = small_batch(240, [500, 123, 64, 1], Hq=14, Hkv=2, D=128, p=16)
    db = DeviceBatch(b)
    want, _ = oracle_decode(b)
    S, Hq, D = 4, 14, 128
    out = torch.zeros((S, Hq, D), dtype=torch.bfloat16, device="cuda")
    ws = torch.empty(mstar.decode_workspace_bytes(S, Hq, D, 4), dtype=torch.uint8, device="cuda")

    def step():
        db.append()
        mstar.paged_attn_decode(out, db.q_decode, db.pool, db.block_table, db.seq_lens, 500, float(b.scale),
                                num_partitions=4, workspace=ws)

    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        step()
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    first = out.clone()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        step()
    out.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(first.view(torch.int16), out.view(torch.int16))
    check_parity(f64_of(out), want, "graph replay")


def test_decode_config2_bagel_cfg_pairs():
    stats = run_decode_case(W.config2_bagel_cfg_decode(), parts_list=(0, 4), check_f32=False)
    print("cfg2", stats)


def test_merge_attn_states_against_combine():
    """mstar_merge_attn_states against COMBINE incl. empty states and the row map (the cascade decode itself is
    mstar_paged_attn_decode_cascade, tests/test_gpu_cascade.py)."""
    # merge kernel alone: random states, -inf on either or both sides, row map
    rng = np.random.default_rng(9)
    N, D = 37, 128
    oa, ob = rng.standard_normal((N + 5, D)).astype(np.float32), rng.standard_normal((N, D)).astype(np.float32)
    la, lb = rng.standard_normal(N + 5).astype(np.float32) * 3, rng.standard_normal(N).astype(np.float32) * 3
    rmap = rng.permutation(N + 5)[:N].astype(np.int32)
    la[rmap[0]] = -np.inf
    lb[1] = -np.inf
    la[rmap[2]] = lb[2] = -np.inf
    o = torch.empty((N, D), dtype=torch.float32, device="cuda")
    l = torch.empty(N, dtype=torch.float32, device="cuda")
    cu = lambda a: torch.from_numpy(a).cuda()
    mstar.merge_attn_states(o, cu(oa), cu(la), cu(ob), cu(lb), row_map_a=cu(rmap), lse_out=l)
    got, got_l = f64_of(o), f64_of(l)
    for r in range(N):
        m = np.array([la[rmap[r]], lb[r]], dtype=np.float64)
        if np.isneginf(m).all():
            assert not got[r].any() and np.isneginf(got_l[r])
            continue
        keep = ~np.isneginf(m)
        w_out, w_lse = oracle.lse_combine(m[keep], np.ones(int(keep.sum())),
                                          np.stack([oa[rmap[r]], ob[r]]).astype(np.float64)[keep])
        assert np.abs(got[r] - w_out).max() < 1e-5 and abs(got_l[r] - w_lse) < 1e-5


def test_decode_config4_thinker_and_talker():
    print("thinker", run_decode_case(W.config4_thinker(), parts_list=(0,), check_f32=False))
    print("talker", run_decode_case(W.config4_talker(), parts_list=(0,), check_f32=False))


def test_decode_config5_long_context_full_size():
    """The bench configuration: 16 x 32768 tokens, 60 GiB pool, 16 partitions; all 512 rows vs the oracle."""
    free, _ = torch.cuda.mem_get_info()
    pages = 491520
    if free < 70 * (1 << 30):   # smaller pool, same 2.1 GB of K/V, if the box is short of memory
        pages = 65536
    b = W.config5_long_context(num_pages=pages)
    db = DeviceBatch(b)
    db.append()
    out, lse = db.decode(num_partitions=16)
    k, v = compact_pool_after_append(b)
    want, want_lse = oracle.paged_decode(b.q, k, v, b.compact_block_table, b.seq_lens, b.scale)
    print("cfg5", check_parity(f64_of(out), want, "cfg5"))
    assert np.abs(f64_of(lse) - want_lse).max() < 2e-3
    # convex-hull invariant at full scale: every output lies within [min_j V, max_j V] of its kv head
    out64 = f64_of(out)
    V = f64_from_bf16_bits(v[b.compact_block_table[0, :1024]])      # sequence 0: [pages, Hkv, p, D]
    vmin, vmax = V.min(axis=(0, 2)), V.max(axis=(0, 2))
    for h in range(32):
        assert np.all(out64[0, h] <= vmax[h // 4] + 1e-6) and np.all(out64[0, h] >= vmin[h // 4] - 1e-6)


# ----------------------------------------------------------------------------- prefill

def run_prefill_case(b, rows=None, causal=True, layout="HND"):
    """Both prefill kernels (tcgen05/TMEM default, mma.sync diagnostic) against the oracle."""
    db = DeviceBatch(b, layout=layout)
    db.append()
    k, v = compact_pool_after_append(b)
    want, want_lse = oracle.paged_prefill(b.q, b.cu_seqlens_q, k, v, b.compact_block_table, b.seq_lens, b.scale,
                                          causal=causal, rows=rows)
    st = {}
    for mma_sync in (False, True):
        out, lse = db.prefill(causal=causal, mma_sync=mma_sync)
        got, got_lse = f64_of(out), f64_of(lse)
        if rows is not None:
            got, got_lse = got[rows], got_lse[rows]
        what = "%s %s" % (b.name, "mma.sync" if mma_sync else "tcgen05")
        st[what] = check_parity(got, want, what)
        assert np.abs(got_lse - want_lse).max() < 2e-3, what
    return st


@pytest.mark.parametrize("D,p", [(64, 16), (128, 16), (128, 32)])
@pytest.mark.parametrize("G", [1, 4, 7, 8, 12])
def test_prefill_ragged_small(D, p, G):
    lens = [40, 17, 33, 5, 64, 200, 129, 1, 300]
    qls = [40, 1, 16, 5, 3, 127, 129, 1, 17]
    b = small_batch(300 + G, lens, q_lens=qls, Hq=G * 2, Hkv=2, D=D, p=p)
    run_prefill_case(b)
    run_prefill_case(b, causal=False)


@pytest.mark.parametrize("Hkv,G", [(1, 8), (8, 4)])
def test_prefill_kv_head_counts(Hkv, G):
    b = small_batch(270 + Hkv, [300, 140, 64], q_lens=[130, 140, 1], Hq=Hkv * G, Hkv=Hkv, D=128, p=16)
    run_prefill_case(b)


def test_prefill_new_tokens_times_prefix_matrix():
    """n in {1, 2, 127, 128, 129} x P in {0, 1, p-1, p, 2047, 2048} as one ragged batch (SURVEY 8(c) matrix);
    G = 7 packs 18 tokens per Q tile, so full tiles (TMA-store epilogue) and ragged tail tiles both occur."""
    p = 16
    lens, qls = [], []
    for n in (1, 2, 127, 128, 129):
        for P in (0, 1, p - 1, p, 2047, 2048):
            lens.append(P + n)
            qls.append(n)
    b = small_batch(305, lens, q_lens=qls, Hq=14, Hkv=2, D=128, p=p)
    run_prefill_case(b)


def test_prefill_long_block_with_and_without_prefix():
    """n = 1024 with P = 0 and P = 2048 (config-3 extremes), sampled rows incl. first / last rows and tile edges."""
    b = small_batch(306, [1024, 3072], q_lens=[1024, 1024], Hq=14, Hkv=2, D=128, p=16)
    rows = np.unique(np.concatenate([np.arange(0, 40), np.arange(1000, 1064), np.arange(2008, 2048),
                                     np.random.default_rng(5).integers(0, 2048, 64)])).astype(np.int32)
    run_prefill_case(b, rows=rows)
    run_prefill_case(b, rows=rows, causal=False)


def test_prefill_flow_step_bidirectional_block_over_cfg_labels():
    """the denoise step -- a block of latent tokens attends bidirectionally to itself and to
    the cached context of its CFG label (causal = 0); the cfg_img label reads the cond label's context pages by
    reference.  Sampled rows incl. block edges; both kernels."""
    b = W.flow_step_bagel(num_requests=2, n_latent=1024)
    rng = np.random.default_rng(61)
    rows = np.unique(np.concatenate([rng.integers(0, b.total_q, 128), b.cu_seqlens_q[:-1],
                                     b.cu_seqlens_q[1:] - 1])).astype(np.int32)
    run_prefill_case(b, rows=rows, causal=False)
    # labels that share context pages and have equal context length see identical K/V for the context; their
    # outputs differ only through their own latent block, so nothing is bit-identical here -- but the shared
    # pages must not have been written by the append of either label
    db = DeviceBatch(b)
    before = bits_of(db.k_pool[torch.from_numpy(b.block_table[0, :4].astype(np.int64)).cuda()])
    db.append()
    after = bits_of(db.k_pool[torch.from_numpy(b.block_table[0, :4].astype(np.int64)).cuda()])
    assert np.array_equal(before, after)


def test_prefill_deterministic_and_graph_capturable():
    """append + plan + attention (programmatic dependent launch between them) captured in a CUDA graph: replays are
    bit-identical to the eager call, repeated eager calls are bit-identical to each other."""
    b = small_batch(330, [300, 1000, 77], q_lens=[200, 260, 77], Hq=14, Hkv=2, D=128, p=16)
    db = DeviceBatch(b)
    T, Hq, D = b.total_q, 14, 128
    out = torch.zeros((T, Hq, D), dtype=torch.bfloat16, device="cuda")
    ws = torch.empty(mstar.prefill_workspace_bytes(b.num_seqs, T, Hq, D), dtype=torch.uint8, device="cuda")

    def step():
        db.append()
        mstar.paged_attn_prefill(out, db.q, db.cu_seqlens_q, db.pool, db.block_table, db.seq_lens, b.max_q_len,
                                 b.max_seq_len, float(b.scale), causal=True, workspace=ws)

    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        step()
        first = out.clone()
        step()
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    assert torch.equal(first.view(torch.int16), out.view(torch.int16))
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        step()
    for _ in range(2):
        out.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(first.view(torch.int16), out.view(torch.int16))
    k, v = compact_pool_after_append(b)
    want, _ = oracle.paged_prefill(b.q, b.cu_seqlens_q, k, v, b.compact_block_table, b.seq_lens, b.scale)
    check_parity(f64_of(out), want, "prefill graph replay")


def test_prefill_one_token_equals_decode_semantics():
    b = small_batch(310, [1, 17, 33, 100, 700], Hq=8, Hkv=2, D=128)
    db = DeviceBatch(b)
    db.append()
    out_p, _ = db.prefill()
    want, _ = oracle_decode(b)
    check_parity(f64_of(out_p), want, "prefill n=1")


def test_prefill_nhd_layout_and_empty_sequences():
    b = small_batch(320, [50, 0, 30, 16], q_lens=[20, 0, 30, 0], Hq=4, Hkv=2, D=128)
    run_prefill_case(b, layout="NHD")


def test_prefill_config3_sampled_rows():
    b = W.config3_prefill()
    rng = np.random.default_rng(33)
    rows = np.unique(np.concatenate([rng.integers(0, b.total_q, 96),
                                     b.cu_seqlens_q[:-1], b.cu_seqlens_q[1:] - 1,
                                     b.cu_seqlens_q[:-1] + 15, b.cu_seqlens_q[:-1] + 16])).astype(np.int32)
    print("cfg3", run_prefill_case(b, rows=rows))


# ----------------------------------------------------------------------------- errors

def test_hbm_read_probe_sums_its_buffer():
    x = torch.randint(-2 ** 31, 2 ** 31 - 1, (1 << 20,), dtype=torch.int32, device="cuda")
    from paper_2606_12688_b200 import bench_aux
    acc = torch.zeros(1, dtype=torch.int64, device="cuda")
    bench_aux.hbm_read_probe(x, x.numel() * 4, acc)
    torch.cuda.synchronize()
    # the kernel adds per-warp sums that wrap at 32 bits; modulo 2^32 that equals the plain sum of the words
    want = int(x.to(torch.int64).sum().item()) % (1 << 32)
    assert int(acc.item()) % (1 << 32) == want
    with pytest.raises(RuntimeError, match="failed"):
        bench_aux.hbm_read_probe(x, 24)


def test_error_codes():
    b = small_batch(400, [300, 20], Hq=4, Hkv=2, D=64)
    db = DeviceBatch(b)
    out = torch.empty((2, 4, 64), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(mstar.MstarError, match="WORKSPACE_TOO_SMALL"):
        mstar.paged_attn_decode(out, db.q_decode, db.pool, db.block_table, db.seq_lens, 300, 0.125, num_partitions=4,
                                workspace=torch.empty(16, dtype=torch.uint8, device="cuda"))
    with pytest.raises(mstar.MstarError, match="INVALID_ARG"):   # Hq not a multiple of Hkv
        q3 = torch.zeros((2, 3, 64), dtype=torch.bfloat16, device="cuda")
        mstar.paged_attn_decode(torch.empty_like(q3), q3, db.pool, db.block_table, db.seq_lens, 33, 0.125,
                                num_partitions=1)
    with pytest.raises(mstar.MstarError, match="INVALID_ARG"):   # misaligned q
        buf = torch.zeros(2 * 4 * 64 + 8, dtype=torch.bfloat16, device="cuda")
        mstar.paged_attn_decode(out, buf[1:1 + 512].view(2, 4, 64), db.pool, db.block_table, db.seq_lens, 33,
                                0.125, num_partitions=1)
    with pytest.raises(mstar.MstarError, match="INVALID_ARG"):   # non-positive scale
        mstar.paged_attn_decode(out, db.q_decode, db.pool, db.block_table, db.seq_lens, 33, 0.0, num_partitions=1)


@pytest.mark.parametrize("Hq,Hkv,D,p", [(32, 1, 128, 16), (48, 2, 64, 32), (40, 2, 128, 32), (64, 1, 128, 16)])
def test_decode_more_than_16_heads_per_kv_head(Hq, Hkv, D, p):
    """Hq / Hkv = 32, 24, 20, 64: the group is split into sub-groups of at most 16 heads (2 x 16, 2 x 12, 2 x 10, 4 x 16), each a
    stream of its own over the same K/V; every partition mode."""
    b = small_batch(470 + Hq, [1, 65, 700, 0, 129, 2300, 64], Hq=Hq, Hkv=Hkv, D=D, p=p)
    db = DeviceBatch(b)
    db.append()
    k, v = compact_pool_after_append(b)
    want, want_lse = oracle.paged_decode(decode_q(b), k, v, b.compact_block_table, b.seq_lens, b.scale)
    for parts in (0, 1, 3, 16):
        out, lse = db.decode(num_partitions=parts)
        check_parity(f64_of(out), want, "G=%d parts=%d" % (Hq // Hkv, parts))
        got = f64_of(lse)
        fin = np.isfinite(want_lse)
        assert np.array_equal(np.isneginf(got), np.isneginf(want_lse))
        assert np.abs(got[fin] - want_lse[fin]).max(initial=0.0) < 2e-3


def test_decode_prime_group_size_above_16():
    """Hq / Hkv = 17 has no divisor that leaves sub-groups of 2 .. 16 heads: every head becomes a stream of its own."""
    b = small_batch(480, [40, 3, 300], Hq=17, Hkv=1, D=128, p=16)
    db = DeviceBatch(b)
    db.append()
    k, v = compact_pool_after_append(b)
    want, _ = oracle.paged_decode(decode_q(b), k, v, b.compact_block_table, b.seq_lens, b.scale)
    for parts in (0, 2):
        out, _ = db.decode(num_partitions=parts)
        check_parity(f64_of(out), want, "G=17 parts=%d" % parts)
