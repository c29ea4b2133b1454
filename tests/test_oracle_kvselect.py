"""Pins for oracle/kvselect.py: pair-by-pair brute force of the needed-key
set, Eq.5 <= Eq.4, the whole-document and N=1 special cases."""
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
