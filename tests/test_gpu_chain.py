"""GPU parity of kv_chain_hash (PAPER.md:L276 chained paged hashing) against
oracle/chain_oracle: 64-bit ids, bit-exact, on the same seeded identity batches."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import chain_oracle as co  # noqa: E402
from paper_2606_31093_b200 import workloads as W  # noqa: E402


@pytest.fixture(scope="module")
def kv():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2606_31093_b200 import kvtier
    return kvtier


@pytest.fixture()
def ctx(kv):
    c = kv.Ctx(0)
    yield c
    torch.cuda.synchronize()
    c.close()


def run(kv, ctx, ident, off, T, roots=None, slack=3):
    d_ident = torch.from_numpy(np.ascontiguousarray(ident).view(np.int64)).cuda()
    n = int((np.diff(off) // T).sum())
    out = torch.full((n + slack,), -1, dtype=torch.int64, device="cuda")
    poff = kv.kv_chain_hash(ctx, d_ident, off, T, out, roots=roots)
    torch.cuda.synchronize()
    got = out.cpu().numpy().view(np.uint64)
    assert (got[n:] == np.uint64(2**64 - 1)).all(), "wrote past the last id"
    return got[:n], poff


@pytest.mark.parametrize("T", [16, 64, 1, 5, 33])
@pytest.mark.parametrize("seed,S,lo,hi", [(0, 64, 512, 16384), (1, 7, 1, 300), (2, 200, 16, 700)])
def test_chain_hash_equals_oracle(kv, ctx, T, seed, S, lo, hi):
    wb = W.identity_batch(seed=seed, n_sessions=S, lo=lo, hi=hi)
    want, wpoff = co.chain_batched(wb.ident, wb.tok_offsets, T)
    got, poff = run(kv, ctx, wb.ident, wb.tok_offsets, T)
    assert np.array_equal(poff, wpoff)
    assert np.array_equal(got, want)
    roots = np.random.default_rng(seed).integers(0, 2**64, size=S, dtype=np.uint64)
    want_r, _ = co.chain_batched(wb.ident, wb.tok_offsets, T, roots)
    got_r, _ = run(kv, ctx, wb.ident, wb.tok_offsets, T, roots=roots)
    assert np.array_equal(got_r, want_r)
    assert not np.array_equal(got_r, got) or got.size == 0


def test_config3_session_and_config4_batch_shapes(kv, ctx):
    """The paper-shaped inputs: one 50-turn session's 46k-token history (2,875 ids, one long chain) and
    the 64-request batch of config 4 (288,990 tokens, 18,059 whole pages)."""
    turns = W.session_turns(seed=0)
    one = W.identity_batch(seed=3, lens=[turns[-1].cum_tokens])
    got, poff = run(kv, ctx, one.ident, one.tok_offsets, 16)
    assert poff.tolist() == [0, turns[-1].cum_tokens // 16]
    assert np.array_equal(got, co.chain(one.ident, 16))
    c4 = W.batch_case(seed=0)
    wb = W.identity_batch(seed=4, lens=c4.lens)
    got, poff = run(kv, ctx, wb.ident, wb.tok_offsets, 16)
    want, wpoff = co.chain_batched(wb.ident, wb.tok_offsets, 16, threads=8)
    assert np.array_equal(poff, wpoff) and np.array_equal(got, want)
    # cross-session reuse: sessions that copied a prefix of session 0 share its leading ids
    for s in np.nonzero(wb.shared_prefix)[0]:
        k = min(int(wb.shared_prefix[s]) // 16, int(poff[1] - poff[0]), int(poff[s + 1] - poff[s]))
        assert np.array_equal(got[poff[s]:poff[s] + k], got[:k])


@pytest.mark.parametrize("T", [16, 5])
def test_thousands_of_ragged_sessions(kv, ctx, T):
    """The two-launch path of large batches (digests of all pages at once, then a warp per session along the chain) on
    1,500 sessions of very unequal length -- a tenth empty, a tenth shorter than a page, one far longer than the rest --
    with and without per-session roots, against the oracle."""
    rng = np.random.default_rng(1500 + T)
    S = 1500
    lens = np.floor(np.exp(rng.uniform(np.log(16), np.log(4000), size=S))).astype(np.int64)
    kind = rng.random(S)
    lens[kind < 0.1] = 0
    sub = (kind >= 0.1) & (kind < 0.2)
    lens[sub] = rng.integers(1, T, size=int(sub.sum()))
    lens[777] = 20000
    off = np.zeros(S + 1, dtype=np.int64)
    np.cumsum(lens, out=off[1:])
    ident = rng.integers(0, 2**64, size=int(off[-1]), dtype=np.uint64)
    want, wpoff = co.chain_batched(ident, off, T, threads=8)
    got, poff = run(kv, ctx, ident, off, T)
    assert np.array_equal(poff, wpoff) and np.array_equal(got, want)
    assert int((np.diff(poff) == 0).sum()) >= 250  # the empty and sub-page sessions yield no ids
    roots = rng.integers(0, 2**64, size=S, dtype=np.uint64)
    want_r, _ = co.chain_batched(ident, off, T, roots, threads=8)
    got_r, _ = run(kv, ctx, ident, off, T, roots=roots)
    assert np.array_equal(got_r, want_r)


def test_empty_sessions_tails_and_offsets_not_at_zero(kv, ctx):
    rng = np.random.default_rng(9)
    ident = rng.integers(0, 2**64, size=500, dtype=np.uint64)
    off = np.array([7, 7, 22, 23, 23, 300, 500], dtype=np.int64)  # first session starts at token 7
    want, wpoff = co.chain_batched(ident, off, 16)
    got, poff = run(kv, ctx, ident, off, 16)
    assert np.array_equal(poff, wpoff) and np.array_equal(got, want)
    assert poff.tolist() == [0, 0, 0, 0, 0, 17, 29]
    # the worked value of tests/test_chain_oracle_pins.py (identity 0x61, T = 1, root 0)
    got, _ = run(kv, ctx, np.array([0x61], dtype=np.uint64), [0, 1], 1, roots=[0])
    assert got.tolist() == co.chain_py([0x61], 1, root=0)


def test_errors_write_nothing_and_capture(kv, ctx):
    ident = torch.zeros(64, dtype=torch.int64, device="cuda")
    out = torch.full((4,), -1, dtype=torch.int64, device="cuda")
    with pytest.raises(kv.KvError) as ei:
        kv.kv_chain_hash(ctx, ident, [0, 64], 8, out, out_capacity=4)  # needs 8 ids
    assert ei.value.status == kv.KV_ERR_SIZE
    torch.cuda.synchronize()
    assert (out == -1).all()
    # up to 128 sessions the tables ride in the kernel parameters: two self-contained launches, capturable;
    # identities are re-read at every replay
    wb = W.identity_batch(seed=8, n_sessions=100, lo=16, hi=300)
    d_ident = torch.from_numpy(wb.ident.view(np.int64)).cuda()
    n = int((np.diff(wb.tok_offsets) // 16).sum())
    outg = torch.zeros(n, dtype=torch.int64, device="cuda")
    side = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        kv.kv_chain_hash(ctx, d_ident, wb.tok_offsets, 16, outg, stream=side)
    for rep in range(2):
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(outg.cpu().numpy().view(np.uint64), co.chain_batched(wb.ident, wb.tok_offsets, 16)[0])
        wb.ident[::7] ^= np.uint64(rep + 1)  # new identities, same graph
        d_ident.copy_(torch.from_numpy(wb.ident.view(np.int64)))
    # more sessions than fit the parameters: refused under capture, nothing enqueued
    big = W.identity_batch(seed=9, n_sessions=129, lo=16, hi=40)
    d_big = torch.from_numpy(big.ident.view(np.int64)).cuda()
    out_big = torch.full((int((np.diff(big.tok_offsets) // 16).sum()),), -1, dtype=torch.int64, device="cuda")
    g2 = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g2, stream=side):
        with pytest.raises(kv.KvError) as ei:
            kv.kv_chain_hash(ctx, d_big, big.tok_offsets, 16, out_big, stream=side)
        assert ei.value.status == kv.KV_ERR_CAPTURE
        ident.add_(0)  # a graph needs at least one node
    torch.cuda.synchronize()
    assert (out_big == -1).all()
    got, _ = run(kv, ctx, big.ident, big.tok_offsets, 16)  # live, through the pinned ring
    assert np.array_equal(got, co.chain_batched(big.ident, big.tok_offsets, 16)[0])


def test_incremental_turns_continue_the_chain(kv, ctx):
    """A 50-turn session hashed turn by turn (each call: only the turn's new whole pages, root = the last id so
    far) gives the ids of the whole history hashed at once -- and both equal the oracle's."""
    turns = W.session_turns(seed=0)
    wb = W.identity_batch(seed=6, lens=[turns[-1].cum_tokens])
    T = 16
    want = co.chain(wb.ident, T)
    got_all, _ = run(kv, ctx, wb.ident, wb.tok_offsets, T)
    assert np.array_equal(got_all, want)
    pieces, done, root = [], 0, kv.KV_CHAIN_ROOT
    for tn in turns:
        n_pages = tn.cum_tokens // T
        if n_pages == done:
            continue
        seg = wb.ident[done * T:n_pages * T]
        ids, _ = run(kv, ctx, seg, [0, seg.size], T, roots=[root])
        pieces.append(ids)
        root, done = int(ids[-1]), n_pages
    assert np.array_equal(np.concatenate(pieces), want)
