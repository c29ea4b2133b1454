"""Host planner / rank layout / KV statistics of libfcp against the oracle: BIT-EXACT
(SURVEY.md section 8(c2), 8(c3)).  No GPU needed."""
import numpy as np
import pytest

import fcp_inputs
from oracle import kvselect as KV
from oracle import planner as P
from test_oracle_planner import parse_golden, random_inputs


def assert_same_plan(fcp, d, N, r_ppm, strategy, align=1):
    want = P.plan(d, N, r_ppm, strategy, align)
    got = fcp.Plan(d, N, r_ppm, strategy, align)
    assert got.shards() == [tuple(s) for s in want.shards]
    assert got.per_doc() == list(want.per_doc)
    st, kst = got.stats(), KV.kv_stats(want)
    loads = P.rank_loads(want)
    assert st["n_ranks"] == N and st["n_docs"] == len(d) and st["n_shards"] == len(want.shards)
    assert st["n_passes"] == len(want.pass_ratios)
    assert st["context_len"] == sum(d) and st["tokens_per_rank"] == sum(d) // N
    assert (st["max_load"], st["sum_load"]) == (max(loads), sum(loads))
    assert st["imbalance_ppm"] == P.imbalance_ppm(want)
    assert (st["eq4_tokens"], st["eq5_tokens"]) == (kst.eq4_tokens, kst.eq5_tokens)
    assert st["max_remote_tokens"] == max(kst.remote) and st["sum_remote_tokens"] == sum(kst.remote)
    assert st["max_gathered_tokens"] == max(kst.gathered)
    assert st["sum_gathered_tokens"] == sum(kst.gathered)
    for r in range(N):
        rs = got.rank_stats(r)
        assert rs["load"] == loads[r] and rs["n_kv"] == kst.gathered[r]
        assert rs["remote_tokens"] == kst.remote[r] and rs["nonlast_tokens"] == kst.nonlast[r]
        lay, olay = got.rank_layout(r), KV.rank_layout(want, r)
        for key in ("cu_seqlens_q", "q_pos_off", "shard_seg", "cu_seqlens_k", "kv_src_start", "kv_len"):
            assert lay[key].dtype == np.int32
            assert lay[key].tolist() == getattr(olay, key).tolist(), key
        assert np.array_equal(lay["q_token_index"], KV.q_token_index(want, r))
        assert np.array_equal(lay["kv_token_index"], KV.gather_index(want, r))
    return want, got


@pytest.mark.parametrize("case", parse_golden(), ids=lambda c: c["name"])
def test_worked_examples(fcp, case):
    assert_same_plan(fcp, case["d"], case["n"], case["r_ppm"], 0, case["align"])


def test_random_small(fcp):
    for d, N, r_ppm, strategy in random_inputs(11, 300):
        assert_same_plan(fcp, d, N, r_ppm, strategy)


@pytest.mark.parametrize("name", ["tiny", "8b", "longtail", "short", "70b", "fig3a", "fig3b"])
def test_bench_configs(fcp, name):
    cfg = fcp_inputs.CONFIGS[name]
    for seed in (0, 1):
        d = fcp_inputs.doc_lengths(name, seed)
        assert sum(d) == cfg.C
        for strategy in (0, 1, 2, 3):
            assert_same_plan(fcp, d, cfg.N, 1_050_000, strategy)


def test_tile_aligned_variant(fcp):
    """fcp_plan_opts.align_tokens: bit-exact against oracle.planner.plan(...,
    align=A) on random inputs and on the bench recipes with A = 128; 0 and 1 are Algorithm 1
    itself; a negative value is INVALID_ARG."""
    for d, N, r_ppm, strategy in random_inputs(31, 250):
        for A in (2, 4, 16):
            assert_same_plan(fcp, d, N, r_ppm, strategy, A)
        assert fcp.Plan(d, N, r_ppm, strategy, 0).shards() == fcp.Plan(d, N, r_ppm, strategy, 1).shards() \
            == [tuple(s) for s in P.plan(d, N, r_ppm, strategy).shards]
    for name in ("8b", "longtail", "short", "70b"):
        cfg = fcp_inputs.CONFIGS[name]
        for seed in (0, 1):
            for strategy in (0, 1):
                assert_same_plan(fcp, fcp_inputs.doc_lengths(name, seed), cfg.N, 1_050_000, strategy, 128)
    with pytest.raises(fcp.FcpError) as e:
        fcp.Plan([8, 8], 2, align=-1)
    assert e.value.status == -1


def test_sched_info_counts_useful_pairs(fcp):
    """The schedule's mask-aware pair count equals the rank's sum of W."""
    for name in ("tiny", "8b", "short"):
        cfg = fcp_inputs.CONFIGS[name]
        d = fcp_inputs.doc_lengths(name, 0)
        want = P.plan(d, cfg.N)
        got = fcp.Plan(d, cfg.N)
        loads = P.rank_loads(want)
        for r in range(cfg.N):
            info = got.sched(r, cfg.Hq, cfg.Hkv, cfg.D).info()
            assert info["useful_pairs"] == loads[r]
            assert info["n_q"] == cfg.C // cfg.N
            lay = KV.rank_layout(want, r)
            # every (q tile, kv tile) pair with at least one visible element, counted directly
            fwd = 0
            for i in range(len(lay.q_pos_off)):
                a, b = int(lay.cu_seqlens_q[i]), int(lay.cu_seqlens_q[i + 1])
                p = int(lay.q_pos_off[i])
                for r0 in range(0, b - a, 128):
                    rows = min(128, b - a - r0)
                    fwd += (p + r0 + rows - 1) // 128 + 1
            assert info["fwd_kv_tiles"] == fwd * cfg.Hq


def test_per_seq_random_and_errors(fcp):
    """Per-Seq baseline plan (strategy 3): bit-exact plan, layout and statistics
    against the oracle on random inputs; C % 2N != 0 is INVALID_ARG on both sides."""
    rng = np.random.default_rng(21)
    for _ in range(200):
        N = int(rng.integers(1, 9))
        n = int(rng.integers(1, 9))
        d = [int(x) for x in rng.integers(1, 300, size=n)]
        d[-1] += (-sum(d)) % (2 * N)
        assert_same_plan(fcp, d, N, 1_050_000, 3)
    with pytest.raises(fcp.FcpError) as e:
        fcp.Plan([10, 4], 2, strategy=3)
    assert e.value.status == -1
    with pytest.raises(ValueError):
        P.plan([10, 4], 2, strategy=3)


def test_piece_layouts_match_oracle(fcp):
    """Local / prefix split (include/fcp.h section 2b): layouts, token index
    lists and remote counts bit-exact against oracle/kvselect.piece_*; the two schedules' useful
    pairs are the two terms of W(p, s) and add up to the unsplit schedule's."""
    cases = list(random_inputs(21, 40))
    cases += [(fcp_inputs.doc_lengths(n, 0), fcp_inputs.CONFIGS[n].N, 0, 0) for n in ("tiny", "8b")]
    for d, N, r_ppm, strategy in cases:
        want = P.plan(d, N, r_ppm or P.DEFAULT_R_PPM, strategy)
        got = fcp.Plan(d, N, r_ppm, strategy)
        for r in range(N):
            full = got.rank_stats(r)
            pairs = {}
            for piece, opiece in ((fcp.PIECE_LOCAL, KV.PIECE_LOCAL), (fcp.PIECE_PREFIX, KV.PIECE_PREFIX)):
                olay = KV.piece_layout(want, r, opiece)
                lay = got.rank_layout(r, piece)
                for key in ("cu_seqlens_q", "q_pos_off", "shard_seg", "cu_seqlens_k", "kv_src_start",
                            "kv_len"):
                    assert lay[key].tolist() == getattr(olay, key).tolist(), key
                assert np.array_equal(lay["q_token_index"], KV.q_token_index(want, r))
                assert np.array_equal(lay["kv_token_index"], KV.piece_gather_index(want, r, opiece))
                rs = got.rank_stats(r, piece)
                assert rs["n_segs"] == rs["n_shards"] == full["n_shards"]
                assert rs["n_q"] == full["n_q"] and rs["n_kv"] == int(olay.kv_len.sum())
                assert rs["remote_tokens"] == KV.piece_remote_tokens(want, r, opiece)
                assert rs["load"] == full["load"]
                if len(d) <= 16 or r == 0:
                    pairs[piece] = got.sched(r, 4, 2, 64, piece).info()
            if pairs:
                mine = [s for s in want.shards if s.rank == r]
                assert pairs[fcp.PIECE_LOCAL]["useful_pairs"] == sum(s.len * (s.len + 1) // 2 for s in mine)
                assert pairs[fcp.PIECE_PREFIX]["useful_pairs"] == sum(s.start * s.len for s in mine)
                assert pairs[fcp.PIECE_LOCAL]["n_q_pad"] == pairs[fcp.PIECE_PREFIX]["n_q_pad"] \
                    == got.sched(r, 4, 2, 64).info()["n_q_pad"]
    with pytest.raises(fcp.FcpError):
        got.rank_stats(0, 3)
    with pytest.raises(fcp.FcpError):
        got.sched(0, 4, 2, 64, piece=7)
