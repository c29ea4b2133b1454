"""Pins for oracle/kvselect.py: pair-by-pair brute force of the needed-key
set, Eq.5 <= Eq.4, the whole-document and N=1 special cases."""
import pytest
import numpy as np

from oracle import planner as P
from oracle import kvselect as KV
from test_oracle_planner import random_inputs


def needed_keys_bruteforce(pl, rank):
    """{global key index : some query token on `rank` attends to it}, built pair by pair from
    the document mask: query t of doc k sees keys 0..t of doc k."""
    off = [0]
    for x in pl.d:
        off.append(off[-1] + x)
    need = set()
    for s in pl.shards:
        if s.rank != rank:
            continue
        for t in range(s.start, s.start + s.len):
            for j in range(0, t + 1):
                need.add(off[s.doc] + j)
    return need


def test_gather_list_is_exactly_the_needed_set():
    for d, N, r_ppm, strategy in random_inputs(3, 120):
        pl = P.plan(d, N, r_ppm, strategy)
        owner = KV.owner_of_tokens(pl)
        assert (owner >= 0).all()
        st = KV.kv_stats(pl)
        for r in range(N):
            idx = KV.gather_index(pl, r)
            need = needed_keys_bruteforce(pl, r)
            assert idx.dtype == np.int32
            assert list(idx) == sorted(need)              # nothing missing, nothing unused
            assert st.gathered[r] == len(need)
            assert st.remote[r] == sum(1 for g in need if owner[g] != r)
            # the rank's own query tokens are all inside its gathered set
            assert set(KV.q_token_index(pl, r).tolist()) <= need
        assert st.eq5_tokens <= st.eq4_tokens             # each rank holds only C/N tokens
        assert st.eq4_tokens == (sum(d) // N) * (N - 1)


def test_eq5_counts_only_non_last_shards():
    pl = P.plan([512, 256, 128, 128], 2)
    st = KV.kv_stats(pl)
    # rank0 holds (0,0,128) (1,0,64) non-last + last shards (0,384,128) (1,192,64) (2,0,128)
    assert st.nonlast == (192, 384)
    assert st.eq5_tokens == 384 and st.eq4_tokens == 512   # 25 % saving


def test_whole_documents_need_no_exchange():
    pl = P.plan([5] * 8, 4)
    st = KV.kv_stats(pl)
    assert st.eq5_tokens == 0 and st.remote == (0, 0, 0, 0) and st.gathered == (10,) * 4


def test_single_rank():
    pl = P.plan([7, 3, 9], 1)
    st = KV.kv_stats(pl)
    assert st.remote == (0,) and st.gathered == (19,) and st.eq4_tokens == 0 == st.eq5_tokens
    assert list(KV.gather_index(pl, 0)) == list(range(19))


def test_rank_layout_tiny():
    pl = P.plan([512, 256, 128, 128], 2)
    lay = KV.rank_layout(pl, 0)
    assert list(lay.cu_seqlens_q) == [0, 128, 256, 320, 384, 512]
    assert list(lay.q_pos_off) == [0, 384, 0, 192, 0]
    assert list(lay.shard_seg) == [0, 0, 1, 1, 2]
    assert list(lay.cu_seqlens_k) == [0, 512, 768, 896]
    assert list(lay.kv_src_start) == [0, 512, 768]
    lay = KV.rank_layout(pl, 1)
    assert list(lay.kv_src_start) == [0, 512, 896] and list(lay.kv_len) == [384, 192, 128]
    # layout and gather index describe the same buffer
    for r in range(2):
        lay = KV.rank_layout(pl, r)
        idx = np.concatenate([np.arange(s, s + l) for s, l in zip(lay.kv_src_start, lay.kv_len)])
        assert (idx == KV.gather_index(pl, r)).all()


def test_scatter_add_is_the_inverse_of_the_gather_brute_force():
    """kvselect.scatter_add pinned by a token-by-token loop: every gathered row lands on the
    global token it was gathered from, rows of different ranks that hit the same token add up,
    tokens no rank gathered stay untouched."""
    rng = np.random.default_rng(3)
    d = [37, 5, 20, 2]
    for N, strategy in ((2, 0), (4, 1), (1, 2)):
        pl = P.plan(d, N, strategy=strategy)
        C = sum(d)
        want = np.zeros((C, 2, 3))
        got = np.zeros((C, 2, 3))
        touched = np.zeros(C, dtype=int)
        for r in range(N):
            gi = KV.gather_index(pl, r)
            part = rng.standard_normal((len(gi), 2, 3))
            KV.scatter_add(pl, r, part, got)
            for row, tok in enumerate(gi):          # brute force
                want[tok] += part[row]
                touched[tok] += 1
        assert np.array_equal(got, want)
        # every token is gathered by its owner at least (a token sees itself)
        assert (touched >= 1).all()
    with pytest.raises(ValueError):
        KV.scatter_add(pl, 0, np.zeros((1, 2, 3)), np.zeros((C, 2, 3)))


def test_scatter_add_of_rank_gradients_equals_per_document_gradient():
    """PAPER.md:109/204 + north_star invariance: sum over ranks of scatter_add(dk_r, dv_r) is the
    gradient of running every document as its own causal attention (no sharding at all)."""
    from oracle import attention as OA
    rng = np.random.default_rng(5)
    d, N, H, D = [24, 9, 15], 2, 2, 4
    C = sum(d)
    Q, K, V, dO = (rng.standard_normal((C, H, D)) for _ in range(4))
    scale = 0.5
    pl = P.plan(d, N)
    dK, dV = np.zeros_like(K), np.zeros_like(V)
    for r in range(N):
        lay = KV.rank_layout(pl, r)
        qi, gi = KV.q_token_index(pl, r), KV.gather_index(pl, r)
        args = (lay.cu_seqlens_q, lay.q_pos_off, lay.shard_seg, lay.cu_seqlens_k, scale)
        o, lse = OA.rank_fwd(Q[qi], K[gi], V[gi], *args)
        _, dk, dv = OA.rank_bwd(Q[qi], K[gi], V[gi], o, lse, dO[qi], *args)
        KV.scatter_add(pl, r, dk, dK)
        KV.scatter_add(pl, r, dv, dV)
    off = 0
    for n in d:                                     # each document on its own: one shard, p = 0
        one = (np.array([0, n]), np.array([0]), np.array([0]), np.array([0, n]), scale)
        sl = slice(off, off + n)
        o, lse = OA.rank_fwd(Q[sl], K[sl], V[sl], *one)
        _, dk, dv = OA.rank_bwd(Q[sl], K[sl], V[sl], o, lse, dO[sl], *one)
        assert np.abs(dK[sl] - dk).max() < 1e-12 and np.abs(dV[sl] - dv).max() < 1e-12
        off += n


# ------------------------------------------------------------------ local / prefix split
def visible_pairs_bruteforce(pl, rank):
    """{(global query token, global key token)} of one rank, pair by pair from the document
    mask."""
    off = KV.doc_offsets(pl.d)
    pairs = set()
    for s in pl.shards:
        if s.rank == rank:
            for t in range(s.start, s.start + s.len):
                for j in range(t + 1):
                    pairs.add((off[s.doc] + t, off[s.doc] + j))
    return pairs


def piece_pairs(pl, rank, piece):
    """(query, key) pairs a piece computes, read off its varlen descriptors with the layout rule
    of include/fcp.h: row t of shard i sees key j of its segment iff j <= q_pos_off + t, j < len."""
    L = KV.piece_layout(pl, rank, piece)
    qi = KV.q_token_index(pl, rank)
    gi = KV.piece_gather_index(pl, rank, piece)
    pairs = []
    for i in range(len(L.q_pos_off)):
        g = int(L.shard_seg[i])
        k0, k1 = int(L.cu_seqlens_k[g]), int(L.cu_seqlens_k[g + 1])
        for t in range(int(L.cu_seqlens_q[i + 1] - L.cu_seqlens_q[i])):
            for j in range(min(k1 - k0, int(L.q_pos_off[i]) + t + 1)):
                pairs.append((int(qi[L.cu_seqlens_q[i] + t]), int(gi[k0 + j])))
    return pairs


def test_local_and_prefix_pieces_partition_the_visible_pairs():
    for d, N, r_ppm, strategy in random_inputs(11, 60):
        pl = P.plan(d, N, r_ppm, strategy)
        for r in range(N):
            loc = piece_pairs(pl, r, KV.PIECE_LOCAL)
            pre = piece_pairs(pl, r, KV.PIECE_PREFIX)
            assert len(set(loc)) == len(loc) and len(set(pre)) == len(pre)   # nothing twice
            assert not (set(loc) & set(pre))                                 # disjoint
            assert set(loc) | set(pre) == visible_pairs_bruteforce(pl, r)    # complete
            # LOCAL needs nothing from other ranks; PREFIX needs what the unsplit gather needs
            assert list(KV.piece_gather_index(pl, r, KV.PIECE_LOCAL)) == list(KV.q_token_index(pl, r))
            assert KV.piece_remote_tokens(pl, r, KV.PIECE_LOCAL) == 0
            assert KV.piece_remote_tokens(pl, r, KV.PIECE_PREFIX) == KV.kv_stats(pl).remote[r]
            # the pair counts are the two terms of W(p, s) = s(s+1)/2 + p s
            mine = [s for s in pl.shards if s.rank == r]
            assert len(loc) == sum(s.len * (s.len + 1) // 2 for s in mine)
            assert len(pre) == sum(s.start * s.len for s in mine)


def test_piece_layout_worked_example():
    # d = (8, 4), N = 2, all Per-Doc (chunks of 2 and 1): rank 0 holds doc0 [0,2)+[6,8) and
    # doc1 [0,1)+[3,4); rank 1 holds doc0 [2,6) and doc1 [1,3)
    pl = P.plan([8, 4], 2, 1_000_000, P.STRATEGY_ALL_PER_DOC)
    assert [(s.doc, s.start, s.len) for s in pl.shards if s.rank == 0] == \
        [(0, 0, 2), (0, 6, 2), (1, 0, 1), (1, 3, 1)]
    loc = KV.piece_layout(pl, 0, KV.PIECE_LOCAL)
    assert list(loc.cu_seqlens_k) == [0, 2, 4, 5, 6] and list(loc.q_pos_off) == [0, 0, 0, 0]
    assert list(loc.kv_src_start) == [0, 6, 8, 11]
    pre = KV.piece_layout(pl, 0, KV.PIECE_PREFIX)
    assert list(pre.kv_len) == [0, 6, 0, 3] and list(pre.q_pos_off) == [0, 6, 0, 3]
    assert list(pre.kv_src_start) == [0, 0, 8, 8] and list(pre.cu_seqlens_k) == [0, 0, 6, 6, 9]
    assert list(KV.piece_gather_index(pl, 0, KV.PIECE_PREFIX)) == [0, 1, 2, 3, 4, 5, 8, 9, 10]
    assert KV.piece_remote_tokens(pl, 0, KV.PIECE_PREFIX) == 4 + 2      # doc0 [2,6), doc1 [1,3)
    one = KV.piece_layout(pl, 1, KV.PIECE_PREFIX)
    assert list(one.kv_len) == [2, 1] and list(one.shard_seg) == [0, 1]
    with pytest.raises(ValueError):
        KV.piece_layout(pl, 0, 0)
