"""GPU parity on inputs that leave the N(0,1) comfort zone, and on the full-size cases round 1 only sampled.

Every BASELINE config draws Q, K, V ~ N(0,1): logits ~N(0,1), the running max settles within the first KV stage, the
tcgen05 prefill kernel's lazy rescale of O in TMEM never fires, exp2 never underflows, and split-K combine weights stay
within a few orders of magnitude.  The patterns of ``workloads/adversarial.py`` (SURVEY 8(c) pin (vi) and the edge
cases of VERDICT r1) drive exactly those paths: a dominant key in the first / a middle / the last KV stage, a ramp
whose stage maximum grows by 11.5 log2 units per stage (> the lazy-rescale threshold 8 at EVERY stage; the property is
asserted on the fp64 logits in tests/test_adversarial_inputs.py), |logits| up to ~70, all-equal logits.  Same gates as
everywhere (tests/util.py), through the C ABI, against the fp64 oracle.  Needs a B200."""
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest
import torch

import oracle
import paper_2606_12688_b200 as mstar
import workloads as W
from oracle import fp8 as ofp8
from tests import test_gpu_fp8 as tfp8
from tests import test_gpu_parity as tpar
from tests.gpu_util import DeviceBatch, DeviceBatchFp8, f64_of
from tests.util import check_parity, compact_pool_after_append, decode_q

pytestmark = pytest.mark.gpu

KINDS = list(W.ADVERSARIAL_KINDS)


def adv_batch(kind, lens, q_lens, seed, Hq=14, Hkv=2, D=128, p=16, stage=128):
    rng = np.random.default_rng(seed)
    pages = sum((l + p - 1) // p for l in lens)
    b = W.make_batch(rng, "adv", lens, q_lens, Hq, Hkv, D, p, max(2 * pages, 4))
    return W.make_adversarial(b, kind, stage=stage, seed=seed)


# ----------------------------------------------------------------------------- prefill (tcgen05 + mma.sync kernels)

@pytest.mark.parametrize("kind", KINDS)
def test_prefill_adversarial_logits_causal_and_flow_step(kind):
    """Prefixes of 0 / 16 / 800 / 1741 tokens and blocks of 129..700 rows: up to 20 KV stages of 128 per unit, so a
    dominant key or the ramp maximum lands in first, middle and last (diagonal) stages; G = 7 (config-2/3 geometry)."""
    lens = [1200, 700, 300, 129, 2041]
    qls = [400, 700, 284, 129, 300]
    b = adv_batch(kind, lens, qls, seed=500 + KINDS.index(kind))
    tpar.run_prefill_case(b)                    # causal over the cached prefix
    tpar.run_prefill_case(b, causal=False)      # the flow-step mask


@pytest.mark.parametrize("kind", ["dominant_last", "ramp", "huge"])
@pytest.mark.parametrize("G,p", [(1, 32), (8, 16), (16, 16)])
def test_prefill_adversarial_other_group_sizes(kind, G, p):
    b = adv_batch(kind, [900, 260, 131], [500, 260, 3], seed=520 + G, Hq=2 * G, Hkv=2, p=p)
    tpar.run_prefill_case(b)


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("G,p", [(7, 16), (8, 32)])
def test_prefill_adversarial_head_dim_64(kind, G, p):
    """The head_dim-64 instantiation of the tcgen05 kernel (one 64-column half per tile, P V with N = 64, the lazy
    rescale over 64 TMEM columns): every adversarial kind over up to 17 KV stages, causal and flow-step mask."""
    b = adv_batch(kind, [1200, 700, 129, 2100], [400, 700, 129, 260], seed=540 + KINDS.index(kind), Hq=2 * G, Hkv=2,
                  D=64, p=p)
    tpar.run_prefill_case(b)
    tpar.run_prefill_case(b, causal=False)


def test_prefill_ramp_rescales_o_in_tmem_with_fp32_output():
    """The ramp with fp32 output: kernel error alone (bf16 P, lazy rescale of O and l) without output rounding."""
    b = adv_batch("ramp", [1500, 640], [700, 640], seed=530)
    db = DeviceBatch(b)
    db.append()
    k, v = compact_pool_after_append(b)
    want, _ = oracle.paged_prefill(b.q, b.cu_seqlens_q, k, v, b.compact_block_table, b.seq_lens, b.scale)
    out, _ = db.prefill(out_dtype=torch.float32)
    _, rel = check_parity(f64_of(out), want, "ramp f32")
    assert rel <= 6e-3


# ----------------------------------------------------------------------------- decode, bf16 pool

@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("G,p", [(7, 16), (4, 32), (16, 16)])
def test_decode_adversarial_logits(kind, G, p):
    """64-token stages: the ramp moves every row's maximum at every stage; the dominant key of the longest sequence sits
    in the last partition (parts = 4, 16) or the last balanced piece (parts = 0): combine weights differ by > e^40."""
    lens = [2048, 1500, 700, 65, 64, 1, 0]
    b = adv_batch(kind, lens, [min(1, l) for l in lens], seed=600 + KINDS.index(kind), Hq=2 * G, Hkv=2, p=p, stage=64)
    tpar.run_decode_case(b, parts_list=(0, 1, 4, 16), check_f32=(kind in ("ramp", "dominant_last")))


# ----------------------------------------------------------------------------- decode, fp8 pool

@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("G,p", [(7, 16), (4, 32), (16, 16)])
def test_decode_fp8_adversarial_logits(kind, G, p):
    """The fp8 kernel skips the O rescale of a stage when no row's maximum moved (warp vote): the ramp makes every vote
    say "rescale", q = 0 / constant K make every vote after the first say "skip".  Scales 0.03..0.06 keep the ramp's
    K values (|k| <= 8.5) below saturation at 448 * scale; 128-token stages (8 consumer warps)."""
    lens = [2048, 1500, 700, 129, 128, 1, 0]
    b = adv_batch(kind, lens, [min(1, l) for l in lens], seed=700 + KINDS.index(kind), Hq=2 * G, Hkv=2, p=p, stage=128)
    tfp8.run_case(b, parts_list=(0, 1, 4, 16), scale_range=(0.03, 0.06))


@pytest.mark.parametrize("kind", ["dominant_last", "ramp", "q_zero"])
def test_decode_fp8_adversarial_on_the_12_warp_kernel(kind):
    """max_seq_len > 8192 and G <= 8: 12 consumer warps on 192-token stages."""
    lens = [9000, 2112, 193, 1]
    if kind == "ramp":
        lens = [6100, 2112, 193, 1]   # 32 stages of 192 keep the ramp exactly representable
    b = adv_batch(kind, lens, [1] * 4, seed=730, Hq=8, Hkv=2, p=16, stage=192)
    if kind == "ramp":
        # a sequence bound of 9000 selects the 12-warp kernel although the longest sequence has 6100 tokens
        k_scale, v_scale = W.fp8_page_scales(3, b.num_pages, b.num_kv_heads, lo=0.03, hi=0.06)
        db = DeviceBatchFp8(b, k_scale, v_scale)
        db.quantise_store()
        db.append()
        k8, v8, ks, vs = tfp8.oracle_pool(b, k_scale, v_scale)
        want, _ = ofp8.paged_decode_fp8(decode_q(b), k8, v8, ks, vs, b.compact_block_table, b.seq_lens, b.scale)
        for parts in (0, 5):
            out = torch.empty((4, 8, 128), dtype=torch.bfloat16, device="cuda")
            ws = torch.empty(mstar.decode_workspace_bytes(4, 8, 128, max(parts, mstar.decode_auto_partitions(4, 2, 9000))),
                             dtype=torch.uint8, device="cuda")
            mstar.paged_attn_decode_fp8(out, db.q_decode, db.pool, db.block_table, db.seq_lens, 9000, float(b.scale),
                                        num_partitions=parts, workspace=ws)
            check_parity(f64_of(out), want, "fp8 ramp 12 warps parts=%d" % parts)
    else:
        tfp8.run_case(b, parts_list=(0, 5), scale_range=(0.03, 0.06))


# ----------------------------------------------------------------------------- full-size cases

def test_prefill_config3_every_work_unit():
    """configs[2] (the prefill headline) compared on three rows of EVERY Q tile of every (sequence, kv head) work unit
    -- first, last and one seeded row of each 18-token tile (a unit = 2 tiles x 4 kv heads; all 28 heads of a row are
    checked, so every (unit, tile, kv head) is covered) -- plus both kernels on the sequence edges."""
    b = W.config3_prefill()
    G = b.num_q_heads // b.num_kv_heads
    tq = 128 // G
    rng = np.random.default_rng(34)
    rows = []
    for s in range(b.num_seqs):
        r0, n = int(b.cu_seqlens_q[s]), int(b.q_lens[s])
        for t0 in range(0, n, tq):
            t1 = min(n, t0 + tq)
            rows += [r0 + t0, r0 + t1 - 1, r0 + int(rng.integers(t0, t1))]
    rows = np.unique(np.array(rows, dtype=np.int32))
    assert rows.size >= 3 * 8 * 56 - 8 * 57
    db = DeviceBatch(b)
    db.append()
    k, v = compact_pool_after_append(b)
    want, want_lse = oracle.paged_prefill(b.q, b.cu_seqlens_q, k, v, b.compact_block_table, b.seq_lens, b.scale, rows=rows)
    out, lse = db.prefill()
    print("cfg3 every unit (%d rows)" % rows.size, check_parity(f64_of(out)[rows], want, "cfg3 tcgen05"))
    assert np.abs(f64_of(lse)[rows] - want_lse).max() < 2e-3
    edge = np.isin(rows, np.concatenate([b.cu_seqlens_q[:-1], b.cu_seqlens_q[1:] - 1]))
    out2, _ = db.prefill(mma_sync=True)
    check_parity(f64_of(out2)[rows[edge]], want[edge], "cfg3 mma.sync edges")


def test_decode_fp8_config5_long_context_full_size():
    """The fp8 bench entry: 16 x 32768 tokens on the 12-warp kernel, 16 partitions of 2112 tokens, 60 GiB-pool geometry
    (491520 pages); codes bit-exact and all 512 rows vs oracle/fp8.py (the oracle runs one sequence per host thread)."""
    free, _ = torch.cuda.mem_get_info()
    pages = 491520 if free > 50 * (1 << 30) else 65536
    b = W.config5_long_context(num_pages=pages)
    k_scale, v_scale = W.fp8_page_scales(83, b.num_pages, b.num_kv_heads)
    db = DeviceBatchFp8(b, k_scale, v_scale)
    db.quantise_store()
    db.append()
    out, lse = db.decode(num_partitions=16)
    gk, gv = db.store_codes()
    Hkv, p, D = b.num_kv_heads, b.page_size, b.head_dim
    q = decode_q(b)

    def one_sequence(s):
        npg = (int(b.seq_lens[s]) + p - 1) // p
        rows = b.compact_block_table[s, :npg].astype(np.int64)
        ks, vs = k_scale[b.used_pages[rows]], v_scale[b.used_pages[rows]]
        k8 = np.full((npg, Hkv, p, D), 0x7F, dtype=np.uint8)
        v8 = np.full_like(k8, 0x7F)
        ofp8.kv_append_fp8(k8, v8, ks, vs, b.k_store[rows].transpose(0, 2, 1, 3).reshape(-1, Hkv, D),
                           b.v_store[rows].transpose(0, 2, 1, 3).reshape(-1, Hkv, D), np.arange(npg * p, dtype=np.int64))
        t0, n = int(b.cu_seqlens_q[s]), int(b.q_lens[s])
        local = {int(r): i for i, r in enumerate(rows)}
        cs = b.compact_slot_mapping[t0:t0 + n]
        slot = np.array([local[int(c // p)] * p + int(c % p) for c in cs], dtype=np.int64)
        ofp8.kv_append_fp8(k8, v8, ks, vs, b.k_new[t0:t0 + n], b.v_new[t0:t0 + n], slot)
        assert np.array_equal(gk[rows], k8) and np.array_equal(gv[rows], v8), "codes of sequence %d" % s
        o, l = ofp8.paged_decode_fp8(q[s:s + 1], k8, v8, ks, vs, np.arange(npg, dtype=np.int32)[None],
                                     b.seq_lens[s:s + 1], b.scale)
        return o[0], l[0]

    with ThreadPoolExecutor(max_workers=8) as ex:
        res = list(ex.map(one_sequence, range(b.num_seqs)))
    want = np.stack([r[0] for r in res])
    want_lse = np.stack([r[1] for r in res])
    print("cfg5 fp8", check_parity(f64_of(out), want, "cfg5 fp8"))
    assert np.abs(f64_of(lse) - want_lse).max() < 2e-3


# ----------------------------------------------------------------------------- plan reuse, PDL behind a metadata update

def test_prefill_reuse_plan_eager_and_graph():
    """MSTAR_FLAG_PREFILL_REUSE_PLAN: layer 1 builds the plan, layers 2..4 reuse it (the last CTA re-arms the work
    counter): bit-identical to non-reuse calls, eager and in a CUDA graph; the plan header is re-armed (0, 0) after
    every call; a changed batch without the flag rebuilds the plan."""
    b = tpar.small_batch(340, [300, 1000, 77, 500], q_lens=[200, 260, 77, 1], Hq=14, Hkv=2, D=128, p=16)
    db = DeviceBatch(b)
    db.append()
    T, Hq, D = b.total_q, 14, 128
    ws = torch.empty(mstar.prefill_workspace_bytes(b.num_seqs, T, Hq, D), dtype=torch.uint8, device="cuda")
    ws.fill_(0xFF)
    out = torch.zeros((T, Hq, D), dtype=torch.bfloat16, device="cuda")

    def call(reuse, o=out, d=db, bb=b):
        mstar.paged_attn_prefill(o, d.q, d.cu_seqlens_q, d.pool, d.block_table, d.seq_lens, bb.max_q_len,
                                 bb.max_seq_len, float(bb.scale), causal=True, workspace=ws, reuse_plan=reuse)

    call(False)
    torch.cuda.synchronize()
    ref = out.clone()
    hdr = ws[:12].view(torch.int32).cpu().numpy()
    assert hdr[0] == 0 and hdr[1] == 0 and hdr[2] > 0
    for _ in range(3):
        out.zero_()
        call(True)
        torch.cuda.synchronize()
        assert torch.equal(ref.view(torch.int16), out.view(torch.int16))
        hdr = ws[:12].view(torch.int32).cpu().numpy()
        assert hdr[0] == 0 and hdr[1] == 0
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        call(False)
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        call(False)
        call(True)
        call(True)
    out.zero_()
    g.replay()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(ref.view(torch.int16), out.view(torch.int16))
    # a different batch in the same workspace, no flag: the plan is rebuilt
    b2 = tpar.small_batch(341, [640, 64], q_lens=[130, 64], Hq=14, Hkv=2, D=128, p=16)
    db2 = DeviceBatch(b2)
    db2.append()
    out2 = torch.zeros((b2.total_q, Hq, D), dtype=torch.bfloat16, device="cuda")
    call(False, out2, db2, b2)
    k, v = compact_pool_after_append(b2)
    want, _ = oracle.paged_prefill(b2.q, b2.cu_seqlens_q, k, v, b2.compact_block_table, b2.seq_lens, b2.scale)
    check_parity(f64_of(out2), want, "rebuilt plan")


@pytest.mark.parametrize("fp8", [False, True])
def test_decode_behind_a_kernel_that_writes_seq_lens_and_block_table(fp8):
    """The split-K kernel is launched with programmatic stream serialization: a kernel that advances seq_lens and
    fills in the block table (a device-side step advance of a captured decode loop) directly precedes it, eager and
    inside a CUDA graph; the decode must see the new metadata (griddepcontrol.wait precedes every global read)."""
    lens = [700, 64, 333, 1]
    b = tpar.small_batch(350, lens, Hq=14, Hkv=2, D=128, p=16)
    S, Hq, D = 4, 14, 128
    if fp8:
        k_scale, v_scale = W.fp8_page_scales(4, b.num_pages, b.num_kv_heads)
        db = DeviceBatchFp8(b, k_scale, v_scale)
        db.quantise_store()
        db.append()
        k8, v8, ks, vs = tfp8.oracle_pool(b, k_scale, v_scale)
        want, _ = ofp8.paged_decode_fp8(decode_q(b), k8, v8, ks, vs, b.compact_block_table, b.seq_lens, b.scale)
    else:
        db = DeviceBatch(b)
        db.append()
        want, _ = tpar.oracle_decode(b)
    true_lens, true_bt = db.seq_lens.clone(), db.block_table.clone()
    out = torch.zeros((S, Hq, D), dtype=torch.bfloat16, device="cuda")
    ws = torch.empty(mstar.decode_workspace_bytes(S, Hq, D, mstar.decode_auto_partitions(S, 2, 700)), dtype=torch.uint8,
                     device="cuda")
    dec = mstar.paged_attn_decode_fp8 if fp8 else mstar.paged_attn_decode

    def step(parts):
        torch.add(true_lens, 0, out=db.seq_lens)       # written by KERNELS right before the decode ...
        torch.add(true_bt, 0, out=db.block_table)
        dec(out, db.q_decode, db.pool, db.block_table, db.seq_lens, 700, float(b.scale), num_partitions=parts,
            workspace=ws)
        db.seq_lens.fill_(1)               # ... and stale again right after it
        db.block_table.fill_(0)

    for parts in (0, 1, 3):
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            step(parts)
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        check_parity(f64_of(out), want, "eager parts=%d" % parts)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            step(parts)
        for _ in range(3):
            out.zero_()
            g.replay()
        torch.cuda.synchronize()
        check_parity(f64_of(out), want, "graph parts=%d" % parts)
