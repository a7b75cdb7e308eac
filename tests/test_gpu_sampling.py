"""GPU parity of mstar_sample_tokens against oracle/sampling.py (R28).  The sampled token is an integer
decided by floating point (a running sum against u): it is correct when it lies in the oracle's support and u lies in
its fp64 interval of the running sum widened by 1e-5; inputs whose top-k / top-p cut is itself within rounding are not
generated (the generator below redraws them).  Greedy rows and uniform logits are compared exactly."""
import numpy as np
import pytest
import torch

import paper_2606_12688_b200 as mstar
from oracle import sampling as smp

pytestmark = pytest.mark.gpu
DELTA = 1e-5


def unambiguous(lg, T, k, p):
    """True when neither the top-k nor the top-p cut sits within rounding of a tie / the target mass."""
    z = np.sort(lg.astype(np.float64) / T)[::-1]
    V = len(z)
    if 0 < k < V and z[k - 1] - z[k] < 1e-3:
        return False
    if 0 < p < 1:
        kept, _ = smp.support(lg, T, k, 1.0)
        q = np.where(kept, np.exp(lg / T - (lg / T).max()), 0)
        q /= q.sum()
        o = np.argsort(-q, kind="stable")
        cum = np.cumsum(q[o])
        n = int(np.searchsorted(cum, p)) + 1
        if abs(cum[n - 1] - p) < 1e-4 or (n >= 2 and abs(cum[n - 2] - p) < 1e-4):
            return False
        if n < V and q[o[n - 1]] - q[o[n]] < 1e-7 and q[o[n]] > 0:
            return False
    return True


def run(logits, T, K, P, seeds, step, dtype=torch.float32, advance=False, one_cta=False, pad=0):
    B, V = logits.shape
    lg = torch.from_numpy(logits.astype(np.float32)).cuda().to(dtype)
    if pad:   # rows that start off a 16-byte boundary, with a stride that is not a multiple of the vector width
        big = torch.full((B, V + 2 * pad + 1), float("nan"), dtype=dtype, device="cuda")
        big[:, pad:pad + V] = lg
        lg = big[:, pad:pad + V]
    out = torch.full((B,), -1, dtype=torch.int32, device="cuda")
    st = torch.tensor([step], dtype=torch.int64, device="cuda")
    mstar.sample_tokens(out, lg, torch.from_numpy(np.asarray(seeds, dtype=np.int64)).cuda(), st,
                        temperature=torch.from_numpy(np.asarray(T, np.float32)).cuda(),
                        top_k=torch.from_numpy(np.asarray(K, np.int32)).cuda(),
                        top_p=torch.from_numpy(np.asarray(P, np.float32)).cuda(), advance_step=advance,
                        one_cta=one_cta)
    torch.cuda.synchronize()
    return out.cpu().numpy(), lg.float().cpu().numpy().astype(np.float64), int(st.item())


def check_rows(tok, lg64, T, K, P, seeds, step, rows=None):
    """rows: the row numbers the entries had in the call (the Philox counter holds the row); default 0, 1, ..."""
    exact = 0
    for r in range(len(tok)):
        t = int(tok[r])
        assert 0 <= t < lg64.shape[1]
        if T[r] == 0:
            assert t == int(np.argmax(lg64[r]))
            continue
        u = smp.uniform(int(seeds[r]), step, r if rows is None else int(rows[r]))
        ok, lo, hi = smp.cdf_interval(lg64[r], float(np.float32(T[r])), int(K[r]), float(np.float32(P[r])), t)
        assert ok, "row %d: token %d outside the support" % (r, t)
        assert lo - DELTA <= u <= hi + DELTA, "row %d: u = %.9f not in [%.9f, %.9f]" % (r, u, lo, hi)
        exact += t == smp.sample(lg64[r], float(np.float32(T[r])), int(K[r]), float(np.float32(P[r])), u)
    return exact


def make_rows(rng, B, V, sigma=2.0):
    lg = np.zeros((B, V))
    T, K, P = np.zeros(B, np.float32), np.zeros(B, np.int32), np.ones(B, np.float32)
    for r in range(B):
        while True:
            lg[r] = np.float32(rng.normal(0, sigma, V))
            T[r] = np.float32(rng.choice([0.0, 0.5, 0.8, 1.0, 1.7]))
            K[r] = int(rng.choice([0, 0, 1, 5, 50, V - 1, V, V + 7]))
            P[r] = np.float32(rng.choice([1.0, 1.0, 0.95, 0.8, 0.3, 1e-6]))
            if T[r] == 0 or unambiguous(lg[r], float(T[r]), int(K[r]) if K[r] < V else 0, float(P[r])):
                break
    return lg, T, K, P


@pytest.mark.parametrize("V", [1, 2, 33, 1000, 4099])
@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
def test_sample_tokens_random_rows_all_filters(V, dtype):
    rng = np.random.default_rng(100 + V)
    B = 64
    lg, T, K, P = make_rows(rng, B, V)
    if dtype == torch.bfloat16:   # decide ambiguity on the values the kernel sees
        lgb = torch.from_numpy(lg.astype(np.float32)).to(torch.bfloat16).float().numpy().astype(np.float64)
        for r in range(B):
            if T[r] != 0 and not unambiguous(lgb[r], float(T[r]), int(K[r]) if K[r] < V else 0, float(P[r])):
                K[r], P[r] = 0, 1.0
    seeds = rng.integers(0, 2 ** 62, B)
    for step in (0, 1, 2 ** 33 + 5):
        tok, lg64, _ = run(lg, T, K, P, seeds, step, dtype=dtype)
        exact = check_rows(tok, lg64, T, K, P, seeds, step)
        assert exact >= 0.95 * (T != 0).sum()   # away from interval boundaries the token is the oracle's own


@pytest.mark.parametrize("V", [1, 7, 4096, 4099, 8200, 16390, 40001, 151936])
@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
def test_sample_tokens_cluster_kernel_equals_one_cta_kernel(V, dtype):
    """The cluster kernel (1, 2, 4, 8 CTAs per row by vocabulary size; the default) and the one-CTA kernel compute the
    same keys, fixed-point weights and index-order inversion: the same token on rows of every kind -- ties at the
    top-k / top-p cut, -inf entries, a cut among tokens of weight 0, greedy rows, unaligned rows."""
    rng = np.random.default_rng(900 + V)
    B = 24
    lg = np.float32(rng.normal(0, 3.0, (B, V)))
    lg[:, ::5] = np.round(lg[:, ::5] * 4) / 4          # many exact ties
    lg[B // 2:, 1::7] = -np.inf
    lg[3] = 1.25                                       # all equal
    lg[4, :] = -40.0
    lg[4, V // 2] = 0.0                                # every other token has weight 0
    T = np.float32(rng.choice([0.0, 0.3, 0.8, 1.0, 2.5], B))
    K = rng.choice([0, 1, 2, 50, max(1, V // 2), max(1, V - 1), V], B).astype(np.int32)
    P = np.float32(rng.choice([1.0, 0.999, 0.9, 0.5, 1e-6], B))
    T[3], T[4] = 1.0, 1.0
    seeds = rng.integers(0, 2 ** 62, B)
    for step, pad in ((0, 0), (7, 0), (3, 3)):
        a, _, _ = run(lg, T, K, P, seeds, step, dtype=dtype, pad=pad)
        b, _, _ = run(lg, T, K, P, seeds, step, dtype=dtype, pad=pad, one_cta=True)
        assert np.array_equal(a, b), (V, step, pad, np.flatnonzero(a != b), a[a != b], b[a != b])
        assert np.all((a >= 0) & (a < V))


@pytest.mark.parametrize("V", [8 * 49152, 8 * 49152 + 8])
def test_sample_tokens_cluster_capacity_boundary(V):
    """393 216 entries fill the cluster kernel (8 CTAs x 49 152 tokens, 213 KB of shared memory each); one chunk more
    takes the one-CTA kernel.  Same tokens as the forced one-CTA path, valid against the oracle."""
    rng = np.random.default_rng(77)
    B = 4
    lg = np.float32(rng.normal(0, 2.5, (B, V)))
    T = np.array([1.0, 0.7, 0.0, 1.2], np.float32)
    K = np.array([0, 64, 0, 0], np.int32)
    P = np.array([1.0, 1.0, 1.0, 0.85], np.float32)
    for r in range(B):
        if T[r] != 0 and not unambiguous(lg[r].astype(np.float64), float(T[r]), int(K[r]), float(P[r])):
            K[r], P[r] = 0, 1.0
    seeds = rng.integers(0, 2 ** 62, B)
    a, lg64, _ = run(lg, T, K, P, seeds, 5)
    b, _, _ = run(lg, T, K, P, seeds, 5, one_cta=True)
    assert np.array_equal(a, b)
    check_rows(a, lg64, T, K, P, seeds, 5)


def test_sample_tokens_vocab_of_a_real_tokenizer_size():
    """151 936 entries (the Qwen-family vocabulary of the paper's LLM backbones): 16 rows, every filter."""
    rng = np.random.default_rng(7)
    B, V = 16, 151936
    lg = np.float32(rng.normal(0, 3.0, (B, V)))
    T = np.array([0.0, 1.0, 0.7, 1.0, 0.9, 1.3, 0.6, 1.0] * 2, np.float32)
    K = np.array([0, 0, 50, 0, 20, 1000, 0, 1] * 2, np.int32)
    P = np.array([1.0, 1.0, 1.0, 0.9, 0.95, 1.0, 0.5, 1.0] * 2, np.float32)
    for r in range(B):
        if T[r] != 0 and not unambiguous(lg[r].astype(np.float64), float(T[r]), int(K[r]), float(P[r])):
            K[r], P[r] = 0, 1.0
    seeds = rng.integers(0, 2 ** 62, B)
    tok, lg64, _ = run(lg, T, K, P, seeds, 12345)
    check_rows(tok, lg64, T, K, P, seeds, 12345)


def test_sample_tokens_closed_forms_exact():
    """Uniform logits invert to floor(u V); -inf logits never win; top-k = 1 / top-p -> 0 / T -> 0 are the argmax."""
    V, B = 37, 200
    seeds = np.arange(B) + 5
    tok, _, _ = run(np.zeros((B, V)), np.ones(B), np.zeros(B), np.ones(B), seeds, 9)
    want = [int(np.floor(smp.uniform(int(seeds[r]), 9, r) * V)) for r in range(B)]
    assert tok.tolist() == want
    zeros = np.zeros((B, V), np.float32)
    zeros[:, ::2] = -0.0                               # -0 and +0 are equal values: greedy takes index 0
    tok, _, _ = run(zeros, np.zeros(B), np.zeros(B), np.ones(B), seeds, 9)
    assert not tok.any()
    tok, _, _ = run(zeros, np.ones(B), np.zeros(B), np.ones(B), seeds, 9)
    assert tok.tolist() == want                        # and sampling sees uniform logits
    rng = np.random.default_rng(3)
    lg = np.float32(rng.normal(0, 2, (B, V)))
    lg[:, ::2] = -np.inf
    tok, _, _ = run(lg, np.ones(B), np.zeros(B), np.ones(B), seeds, 1)
    assert np.all(tok % 2 == 1)
    am = np.argmax(np.float32(rng.normal(0, 2, (B, V))), axis=1)
    lg2 = np.full((B, V), -3.0, np.float32)
    lg2[np.arange(B), am] = 4.0
    for T, K, P in ((1.0, 1, 1.0), (1.0, 0, 1e-6), (1e-3, 0, 1.0), (0.0, 0, 1.0)):
        tok, _, _ = run(lg2, np.full(B, T), np.full(B, K), np.full(B, P), seeds, 2)
        assert np.array_equal(tok, am)


def test_sample_tokens_frequencies_follow_the_softmax():
    """4096 rows with the same logits and different seeds: chi-square against the softmax computed here."""
    rng = np.random.default_rng(21)
    V, B, T = 16, 4096, 0.8
    row = np.float32(rng.normal(0, 1.2, V))
    pr = np.exp(row.astype(np.float64) / np.float32(T))
    pr /= pr.sum()
    tok, _, _ = run(np.tile(row, (B, 1)), np.full(B, T), np.zeros(B), np.ones(B), rng.integers(0, 2 ** 62, B), 3)
    cnt = np.bincount(tok, minlength=V)
    chi2 = float((((cnt - B * pr) ** 2) / (B * pr)).sum())
    assert chi2 < (V - 1) + 5 * np.sqrt(2 * (V - 1)) + 5, chi2


def test_sample_tokens_graph_replay_draws_fresh_numbers_and_is_deterministic():
    """Captured once, replayed with the step counter advanced on the device: every replay equals the eager call at
    that step; the same (seed, step) gives the same token."""
    rng = np.random.default_rng(5)
    B, V = 32, 500
    lg = torch.from_numpy(np.float32(rng.normal(0, 2, (B, V)))).cuda()
    seeds = torch.from_numpy(rng.integers(0, 2 ** 62, B)).cuda()
    T = torch.full((B,), 0.9, device="cuda")
    K = torch.full((B,), 40, dtype=torch.int32, device="cuda")
    P = torch.full((B,), 0.9, device="cuda")
    step = torch.zeros(1, dtype=torch.int64, device="cuda")
    out = torch.empty(B, dtype=torch.int32, device="cuda")
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        call = lambda: mstar.sample_tokens(out, lg, seeds, step, temperature=T, top_k=K, top_p=P, advance_step=True)
        call()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            call()
    torch.cuda.synchronize()
    step.zero_()
    replayed = []
    for _ in range(4):
        g.replay()
        torch.cuda.synchronize()
        replayed.append(out.cpu().numpy().copy())
    assert int(step.item()) == 4
    ref = torch.empty_like(out)
    for s in range(4):
        mstar.sample_tokens(ref, lg, seeds, torch.tensor([s], dtype=torch.int64, device="cuda"), temperature=T,
                            top_k=K, top_p=P)
        torch.cuda.synchronize()
        assert np.array_equal(ref.cpu().numpy(), replayed[s])
    assert not np.array_equal(replayed[0], replayed[1])


def test_sample_tokens_error_codes():
    out = torch.empty(4, dtype=torch.int32, device="cuda")
    lg = torch.zeros((4, 10), device="cuda")
    seeds = torch.zeros(4, dtype=torch.int64, device="cuda")
    step = torch.zeros(1, dtype=torch.int64, device="cuda")
    lib = mstar.load_library()
    assert lib.mstar_sample_tokens(out.data_ptr(), lg.data_ptr(), 10, 4, 10, None, None, None, seeds.data_ptr(),
                                   step.data_ptr(), 0, None) == 0
    assert lib.mstar_sample_tokens(out.data_ptr(), lg.data_ptr(), 5, 4, 10, None, None, None, seeds.data_ptr(),
                                   step.data_ptr(), 0, None) == -1      # row_stride < vocab
    assert lib.mstar_sample_tokens(out.data_ptr(), lg.data_ptr(), 10, 4, 10, None, None, None, None,
                                   step.data_ptr(), 0, None) == -1      # no seeds
    assert lib.mstar_sample_tokens(out.data_ptr(), lg.data_ptr(), 10, 4, 10, None, None, None, seeds.data_ptr(),
                                   step.data_ptr(), 64, None) == -1     # unknown flag
    torch.cuda.synchronize()
