"""Host tile schedule of libfcp against a plain restatement of
its definition (include/fcp.h, fcp_sched_get_list): the enumeration of the forward and backward
work items with their mask-skipping tile counts, the cost order and the greedy
longest-processing-time assignment to the persistent CTAs.  BIT-EXACT, no GPU needed.  The
restatement below is written from the header text with a binary heap; the library uses a
counting sort and a bucket queue."""
import heapq

import numpy as np
import pytest

import fcp_inputs

TQ, TK, BQ = 128, 128, 64      # forward q tile, KV tile, backward q tile (rows)


def lpt(items, cost, n_cta):
    """Stable sort by descending cost, then each item to the least loaded CTA (ties: lowest CTA
    index); returns the items grouped by CTA in assignment order and the CTA offsets."""
    order = sorted(range(len(items)), key=lambda i: -cost(items[i]))          # sorted() is stable
    heap = [(0, c) for c in range(n_cta)]
    lists = [[] for _ in range(n_cta)]
    for i in order:
        load, c = heap[0]
        lists[c].append(items[i])
        heapq.heapreplace(heap, (load + cost(items[i]), c))
    off = np.cumsum([0] + [len(l) for l in lists]).astype(np.int32)
    return [it for l in lists for it in l], off


def reference_lists(cu_q, p_off, seg, cu_k, Hq, Hkv, n_cta):
    G = Hq // Hkv
    NQ = 2 if G % 2 == 0 else 1
    ns = len(p_off)
    fwd, pad0, pad = [], [], 0
    for i in range(ns):
        a, ln, p = int(cu_q[i]), int(cu_q[i + 1] - cu_q[i]), int(p_off[i])
        kv0, kvl = int(cu_k[seg[i]]), int(cu_k[seg[i] + 1] - cu_k[seg[i]])
        pad0.append(pad)
        pad += -(-ln // BQ) * BQ
        for r0 in range(0, ln, TQ):
            rows = min(TQ, ln - r0)
            last_vis = min(kvl - 1, p + r0 + rows - 1)       # last key any row of the tile sees
            n_tiles = 0 if last_vis < 0 else last_vis // TK + 1
            for hk in range(Hkv):
                for pk in range(G // NQ):
                    fwd.append((a + r0, rows, kv0, kvl, p + r0, n_tiles, hk * G + pk * NQ, hk))
    bwd, sub = [], []
    for g in range(len(cu_k) - 1):
        kv0, kvl = int(cu_k[g]), int(cu_k[g + 1] - cu_k[g])
        for c0 in range(0, kvl, TK):
            begin, q_tiles = len(sub), 0
            for i in range(ns):
                a, ln, p = int(cu_q[i]), int(cu_q[i + 1] - cu_q[i]), int(p_off[i])
                if seg[i] != g or ln == 0 or p + ln - 1 < c0:
                    continue                                   # no row of the shard sees the tile
                qt0 = max(0, c0 - p) // BQ                     # first 64-row q tile that sees it
                sub.append((a + qt0 * BQ, p + qt0 * BQ, ln - qt0 * BQ, pad0[i] + qt0 * BQ))
                q_tiles += -(-(ln - qt0 * BQ) // BQ)
            for hk in range(Hkv):
                bwd.append((kv0 + c0, min(TK, kvl - c0), c0, hk, begin, len(sub), q_tiles * G, 0))
    fwd, fwd_off = lpt(fwd, lambda x: x[5] + 1, n_cta)
    bwd, bwd_off = lpt(bwd, lambda x: x[6] + 2, n_cta)
    as2d = lambda rows, w: np.array(rows, dtype=np.int32).reshape(-1, w)
    return {"fwd": as2d(fwd, 8), "bwd": as2d(bwd, 8), "sub": as2d(sub, 4), "fwd_cta": fwd_off,
            "bwd_cta": bwd_off}


def check(sched, cu_q, p_off, seg, cu_k, Hq, Hkv):
    got = sched.lists()
    n_cta = len(got["fwd_cta"]) - 1
    assert n_cta >= 1 and len(got["bwd_cta"]) == n_cta + 1
    want = reference_lists(cu_q, p_off, seg, cu_k, Hq, Hkv, n_cta)
    for k in want:
        assert np.array_equal(got[k], want[k]), k
    info = sched.info()
    assert info["n_fwd_items"] == len(want["fwd"]) and info["n_bwd_items"] == len(want["bwd"])
    # properties that do not depend on the restatement: every (q row, query head) is in exactly
    # one forward item, every (key row, kv head) in exactly one backward item; greedy LPT bound
    G = Hq // Hkv
    NQ = 2 if G % 2 == 0 else 1
    n_q, n_kv = int(cu_q[-1]), int(cu_k[-1])
    cover = np.zeros((n_q, Hq), dtype=np.int32)
    for q_row0, q_rows, _, _, _, _, head0, _ in got["fwd"]:
        cover[q_row0:q_row0 + q_rows, head0:head0 + NQ] += 1
    assert (cover == 1).all()
    cover = np.zeros((n_kv, Hkv), dtype=np.int32)
    for kv_row0, kv_rows, _, kv_head, _, _, _, _ in got["bwd"]:
        cover[kv_row0:kv_row0 + kv_rows, kv_head] += 1
    assert (cover == 1).all()
    for items, off, col, extra in ((got["fwd"], got["fwd_cta"], 5, 1), (got["bwd"], got["bwd_cta"], 6, 2)):
        if len(items):
            cost = items[:, col].astype(np.int64) + extra
            loads = np.array([cost[off[c]:off[c + 1]].sum() for c in range(n_cta)])
            assert loads.max() <= cost.sum() / n_cta + cost.max()


@pytest.mark.parametrize("name", ["tiny", "8b", "short", "longtail"])
def test_bench_config_schedules(fcp, name):
    cfg = fcp_inputs.CONFIGS[name]
    plan = fcp.Plan(fcp_inputs.doc_lengths(name, 0), cfg.N)
    for r in sorted({0, cfg.N // 2, cfg.N - 1}):
        lay = plan.rank_layout(r)
        check(plan.sched(r, cfg.Hq, cfg.Hkv, cfg.D), lay["cu_seqlens_q"], lay["q_pos_off"],
              lay["shard_seg"], lay["cu_seqlens_k"], cfg.Hq, cfg.Hkv)


def test_random_plans_and_pieces(fcp):
    rng = np.random.default_rng(5)
    done = 0
    for case in range(60):
        N = int(rng.choice([1, 2, 4, 8]))
        C = N * int(rng.integers(40, 1500))
        d = fcp_inputs.random_doc_lengths(rng, C, 1, int(rng.choice([90, 700, 4000])))
        Hkv = int(rng.choice([1, 2]))
        Hq = Hkv * int(rng.choice([1, 2, 3, 4]))
        try:
            plan = fcp.Plan(d, N, strategy=int(rng.choice([0, 0, 1, 3])))
        except fcp.FcpError:           # a strategy this (C, N) does not admit
            continue
        done += 1
        r = int(rng.integers(0, N))
        for piece in (fcp.PIECE_FULL, fcp.PIECE_LOCAL, fcp.PIECE_PREFIX):
            lay = plan.rank_layout(r, piece)
            check(plan.sched(r, Hq, Hkv, 64, piece), lay["cu_seqlens_q"], lay["q_pos_off"],
                  lay["shard_seg"], lay["cu_seqlens_k"], Hq, Hkv)
    assert done >= 40


def test_explicit_layout_with_empty_and_unseen_parts(fcp):
    """fcp_sched_create on hand-made arrays: an empty shard, a shard whose offset is negative (a
    KV piece that starts after the document's first token), a segment no shard points to and a
    segment longer than any query sees (trailing KV tiles get items with n_iters = 0)."""
    cu_q = np.array([0, 200, 200, 330, 400], dtype=np.int32)
    p_off = np.array([100, 0, -129, 900], dtype=np.int32)
    seg = np.array([0, 0, 1, 3], dtype=np.int32)
    cu_k = np.array([0, 300, 390, 500, 2000], dtype=np.int32)
    sched = fcp.Sched.create(cu_q, p_off, seg, cu_k, 6, 2, 128)
    check(sched, cu_q, p_off, seg, cu_k, 6, 2)
    L = sched.lists()
    assert (L["bwd"][:, 6] == 0).any() and (L["fwd"][:, 5] == 0).any()
