"""GPU parity of mstar_paged_attn_decode_cascade against the oracle's PLAIN decode: the
cascade is a work split, its result is the plain definition (oracle pin:
test_cascade_identity_three_branches_ragged_shared_lens_split_pieces)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_12688_b200 as mstar
import workloads as W
from tests.gpu_util import DeviceBatch, f64_of
from tests.util import check_parity, compact_pool_after_append, decode_q

pytestmark = pytest.mark.gpu


def oracle_decode(b):
    k, v = compact_pool_after_append(b)
    return oracle.paged_decode(decode_q(b), k, v, b.compact_block_table, b.seq_lens, b.scale)


def cfg_batch(seed, shared_r, sfx, B, Hq, Hkv, D, p):
    """Request-major CFG batch: request r shares shared_r[r] tokens among its B branches, branch b adds sfx[r][b]."""
    R = len(shared_r)
    lens = [shared_r[r] + sfx[r][b] for r in range(R) for b in range(B)]
    share = [-1 if b == 0 else r * B for r in range(R) for b in range(B)]
    shared = [shared_r[r] for r in range(R) for b in range(B)]
    rng = np.random.default_rng(seed)
    pages = sum((l + p - 1) // p for l in lens)
    return W.make_batch(rng, "casc", lens, [1] * len(lens), Hq, Hkv, D, p, 2 * pages + 4, share_with=share,
                        shared_tokens=shared)


def run_case(b, B, shared_r, check_f32=True):
    db = DeviceBatch(b)
    db.append()
    want, want_lse = oracle_decode(b)
    out, lse = db.decode_cascade(B, shared_r)
    stats = check_parity(f64_of(out), want, b.name)
    assert np.abs(f64_of(lse) - want_lse).max() < 2e-3
    if check_f32:
        out32, _ = db.decode_cascade(B, shared_r, out_dtype=torch.float32)
        _, r = check_parity(f64_of(out32), want, b.name + " f32")
        assert r <= 6e-3
    return db, out, stats


@pytest.mark.parametrize("B,G,Hkv,D,p", [(2, 7, 4, 128, 16), (3, 7, 2, 128, 16), (3, 4, 2, 64, 32), (2, 8, 1, 128, 32),
                                         (4, 1, 2, 64, 16), (3, 16, 1, 128, 16), (1, 4, 2, 128, 16)])
def test_cascade_small_ragged(B, G, Hkv, D, p):
    """Ragged shared lengths (0, one page, several tiles), suffixes from one token to several tiles; branch groups
    of floor(16 / G): pairs stacked at G = 7 / 8, three at G = 4, two + one for three labels at G = 7, no stacking
    at G = 16, and the degenerate single-branch call."""
    shared_r = [0, p, 4 * p, 640, 64]
    rng = np.random.default_rng(100 + B * 10 + G)
    sfx = [[int(x) for x in rng.choice([1, 2, p - 1, p, p + 1, 63, 64, 65, 200], B)] for _ in shared_r]
    b = cfg_batch(5 + G, shared_r, sfx, B, G * Hkv, Hkv, D, p)
    run_case(b, B, shared_r)


def test_cascade_equals_plain_on_unshared_batch_and_is_deterministic():
    """shared_lens = 0 everywhere: only suffix streams; the call is then the plain decode's definition.  Two runs
    and a CUDA-graph replay are bit-identical."""
    b = W.make_batch(np.random.default_rng(3), "plain", [100, 1, 700, 64, 33, 257], [1] * 6, 8, 2, 128, 16, 200)
    db, out, _ = run_case(b, 2, [0, 0, 0])
    out2, _ = db.decode_cascade(2, [0, 0, 0])
    assert torch.equal(out.view(torch.int16), out2.view(torch.int16))
    S, Hq, D = b.num_seqs, b.num_q_heads, b.head_dim
    sh = torch.zeros(3, dtype=torch.int32, device="cuda")
    ws = torch.empty(mstar.decode_cascade_workspace_bytes(S, Hq, b.num_kv_heads, D, b.max_seq_len), dtype=torch.uint8,
                     device="cuda")
    og = torch.empty_like(out)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        call = lambda: mstar.paged_attn_decode_cascade(og, db.q_decode, db.pool, db.block_table, db.seq_lens, sh, 2,
                                                       b.max_seq_len, float(b.scale), workspace=ws)
        call()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            call()
    torch.cuda.synchronize()
    og.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out.view(torch.int16), og.view(torch.int16))


def test_cascade_config2_cfg_pairs():
    """BASELINE configs[1]: 32 requests x CFG pair sharing the pages of the first 256 tokens."""
    b = W.config2_bagel_cfg_decode()
    _, _, stats = run_case(b, 2, [256] * 32, check_f32=False)
    print("cascade cfg2", stats)


def test_cascade_three_labels_where_sharing_dominates():
    """16 requests x 3 CFG labels over a shared context of 2048..6144 tokens (the bench's cascade workload), and
    the same with empty sequences mixed in."""
    b, shared = W.cfg_cascade_decode()
    _, _, stats = run_case(b, 3, shared, check_f32=False)
    print("cascade 3 labels", stats)
    assert b.kv_bytes_unique() < 0.5 * b.kv_bytes_logical()


def test_cascade_error_codes():
    b = cfg_batch(1, [16, 16], [[3, 4], [5, 6]], 2, 8, 2, 64, 16)
    db = DeviceBatch(b)
    S, Hq, D = b.num_seqs, b.num_q_heads, b.head_dim
    out = torch.empty((S, Hq, D), dtype=torch.bfloat16, device="cuda")
    sh = torch.tensor([16, 16], dtype=torch.int32, device="cuda")
    ws = torch.empty(mstar.decode_cascade_workspace_bytes(S, Hq, b.num_kv_heads, D, b.max_seq_len), dtype=torch.uint8,
                     device="cuda")
    with pytest.raises(mstar.MstarError):   # one entry per request
        mstar.paged_attn_decode_cascade(out, db.q_decode, db.pool, db.block_table, db.seq_lens, sh[:1], 2,
                                        b.max_seq_len, float(b.scale), workspace=ws)
    with pytest.raises(mstar.MstarError, match="WORKSPACE_TOO_SMALL"):
        mstar.paged_attn_decode_cascade(out, db.q_decode, db.pool, db.block_table, db.seq_lens, sh, 2,
                                        b.max_seq_len, float(b.scale), workspace=ws[:64])
    # raw C ABI: num_seqs not a multiple of n_branches, NULL shared_lens
    import ctypes
    lib = mstar.load_library()
    args = lambda nb, shp: (out.data_ptr(), None, db.q_decode.data_ptr(), ctypes.byref(db.pool.c),
                            db.block_table.data_ptr(), int(db.block_table.stride(0)), db.seq_lens.data_ptr(), shp, S,
                            nb, Hq, int(b.max_seq_len), float(b.scale), 0, ws.data_ptr(), ws.numel(), None)
    assert lib.mstar_paged_attn_decode_cascade(*args(3, sh.data_ptr())) == -1
    assert lib.mstar_paged_attn_decode_cascade(*args(2, None)) == -1
    assert lib.mstar_paged_attn_decode_cascade(*args(0, sh.data_ptr())) == -1
    torch.cuda.synchronize()
