"""Seeded input generators: determinism and the structure DESIGN.md states (no GPU, no oracle)."""
import numpy as np

from paper_2606_31093_b200 import workloads as W


def test_shapes_match_baseline_json():
    assert W.TINY.row_bytes == 4096 and W.TINY.page_bytes == 32768
    q = W.QWEN3_OMNI
    assert q.row_bytes == 16384 and q.tok_bytes == 98304 and q.page_bytes == 1572864
    assert q.L * q.C * q.P * q.row_bytes == 96 << 30


def test_tiny_and_prefix_cases():
    t = W.tiny_case(0)
    assert len(t.src_ids) == len(t.dst_ids) == 37
    assert len(set(t.src_ids)) == 37 and len(set(t.dst_ids)) == 37
    assert np.array_equal(t.src_ids, W.tiny_case(0).src_ids)
    p = W.prefix_case(0)
    assert len(p.src_ids) == 512 and len(set(p.src_ids) | set(p.dst_ids)) == 1024
    assert p.src_ids.dtype == np.int32 and not np.all(np.diff(p.src_ids) > 0)  # fragmented, unsorted


def test_session_turns():
    ts = W.session_turns(0)
    assert len(ts) == 50 and ts[0].n_matched_pages == 0  # turn 1 reloads nothing (the n = 0 no-op)
    c = 0
    for t in ts:
        assert 300 <= t.delta <= 1500 and t.n_matched_pages == c // 16
        assert sum(n for _, n in t.spans) == t.delta
        assert all(256 <= n <= 1024 for k, n in t.spans if k != "text")
        c += t.delta
        assert t.cum_tokens == c
    # seed 0 (DESIGN.md input recipe)
    assert ts[48].cum_tokens == 45687 and ts[49].n_matched_pages == 2855
    assert sum(t.n_matched_pages for t in ts) == 71361


def test_batch_case_matches_survey_numbers():
    b = W.batch_case(0)
    assert int(b.lens.sum()) == 288990 and int(b.req_offsets[-1]) == 18091  # SURVEY.md 8(d) cfg 4
    assert b.lens.min() == 516 and b.lens.max() == 16226
    assert len(set(b.src_ids) | set(b.dst_ids)) == 2 * 18091
    assert np.array_equal(np.diff(b.req_offsets), -(-b.lens // 16))


def test_crossrole_case():
    c = W.crossrole_case(0)
    assert len(c.src_ids) == 32 * 128 and len(c.dst_ids) == 32 * 32
    assert len(set(c.src_ids)) == 4096 and len(set(c.dst_ids)) == 1024
    r = W.crossrole_case(0, ragged=True)
    assert np.all(r.n_tokens < 2048) and np.all(r.n_tokens > 2048 - 64)
    assert np.array_equal(np.diff(r.src_offsets), -(-r.n_tokens // 16)) and np.all(np.diff(r.dst_offsets) == 32)


def test_free_list():
    rng = np.random.default_rng(0)
    fl = W.FreeList(100, rng)
    a = fl.pop(30)
    b = fl.pop(0)
    assert len(a) == 30 and len(b) == 0 and len(set(a)) == 30
    fl.give_back(a)
    assert sorted(fl.free) == list(range(100))


def test_sweep_sizes():
    assert W.sweep_sizes_pages() == [1 << i for i in range(14)]
