"""Pins for oracle/planner.py — checked against what the paper and the mathematics fix, never
against the oracle's own formulas (Eq. 1-3)."""
import itertools
import os

import numpy as np
import pytest

from oracle import planner as P
from oracle import kvselect as KV

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "planner_examples.txt")


def parse_golden(path=GOLDEN):
    cases, cur = [], None
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        tok = line.split()
        if tok[0] == "case":
            cur = {"name": tok[1], "ranks": {}}
            cases.append(cur)
        elif tok[0] == "d":
            cur["d"] = [int(x) for x in tok[1:]]
        elif tok[0] == "n":
            cur["n"], cur["r_ppm"] = int(tok[1]), int(tok[3])
            cur["align"] = int(tok[5]) if len(tok) > 5 else 1
        elif tok[0] == "per_doc":
            cur["per_doc"] = [int(x) for x in tok[1:]]
        elif tok[0] == "rank":
            cur["ranks"][int(tok[1])] = [tuple(int(y) for y in x.split(":")) for x in tok[2:]]
        elif tok[0] == "loads":
            cur["loads"] = [int(x) for x in tok[1:]]
        elif tok[0] == "eq5":
            cur["eq5"], cur["eq4"] = int(tok[1]), int(tok[3])
        elif tok[0] == "remote":
            i = tok.index("gathered")
            cur["remote"] = [int(x) for x in tok[1:i]]
            cur["gathered"] = [int(x) for x in tok[i + 1:]]
    return cases


def brute_pairs(p, s):
    """Unmasked (q,k) pairs of a shard under the causal document mask, counted one by one."""
    return sum(1 for t in range(p, p + s) for j in range(0, t + 1))


def test_W_is_the_pair_count():
    for p in range(0, 9):
        for s in range(1, 9):
            assert P.W(p, s) == brute_pairs(p, s)


@pytest.mark.parametrize("case", parse_golden(), ids=lambda c: c["name"])
def test_worked_examples(case):
    pl = P.plan(case["d"], case["n"], case["r_ppm"], align=case["align"])
    assert list(pl.per_doc) == case["per_doc"]
    for j in range(case["n"]):
        got = [(s.doc, s.start, s.len) for s in pl.shards if s.rank == j]
        assert got == case["ranks"][j]
    assert P.rank_loads(pl) == case["loads"]
    st = KV.kv_stats(pl)
    assert (st.eq5_tokens, st.eq4_tokens) == (case["eq5"], case["eq4"])
    assert list(st.remote) == case["remote"]
    assert list(st.gathered) == case["gathered"]


def test_fig4_ideal_case_any_length():
    for L in (1, 7, 128, 1000):
        pl = P.plan([L, L], 2)
        assert [(s.doc, s.start, s.len, s.rank) for s in pl.shards] == [(0, 0, L, 0), (1, 0, L, 1)]
        assert KV.kv_stats(pl).eq5_tokens == 0
        assert P.imbalance_ppm(pl) == 1_000_000


def random_inputs(seed, count):
    rng = np.random.default_rng(seed)
    for _ in range(count):
        N = int(rng.integers(1, 7))
        n = int(rng.integers(1, 12))
        d = [int(x) for x in rng.integers(1, 60, size=n)]
        pad = (-sum(d)) % N
        if pad:
            d.append(pad)
        r_ppm = int(rng.choice([1_000_000, 1_020_000, 1_050_000, 1_200_000, 2_000_000]))
        strategy = int(rng.integers(0, 3))
        yield d, N, r_ppm, strategy


def check_valid(pl):
    d, N = pl.d, pl.n_ranks
    # Eq. 1: every token of every document on exactly one worker
    cover = [np.zeros(x, dtype=int) for x in d]
    for s in pl.shards:
        assert s.len >= 1 and 0 <= s.start and s.start + s.len <= d[s.doc] and 0 <= s.rank < N
        cover[s.doc][s.start:s.start + s.len] += 1
    assert all((c == 1).all() for c in cover)
    # Eq. 2: exactly C/N tokens per worker
    assert P.rank_tokens(pl) == [sum(d) // N] * N
    # total work is plan independent: sum_shards W = sum_k d_k (d_k+1)/2
    assert sum(P.rank_loads(pl)) == sum(x * (x + 1) // 2 for x in d)
    # canonical order, merged neighbours
    keys = [(s.rank, s.doc, s.start) for s in pl.shards]
    assert keys == sorted(keys)
    for a, b in zip(pl.shards, pl.shards[1:]):
        assert not (a.rank == b.rank and a.doc == b.doc and a.start + a.len == b.start)
    # loads recomputed pair by pair agree with what the loop exit test used
    loads = [0] * N
    for s in pl.shards:
        loads[s.rank] += brute_pairs(s.start, s.len) if s.len * (s.start + s.len) < 5000 \
            else P.W(s.start, s.len)
    assert (max(loads), sum(loads)) == pl.pass_ratios[-1]


def test_invariants_random():
    for d, N, r_ppm, strategy in random_inputs(1, 400):
        pl = P.plan(d, N, r_ppm, strategy)
        check_valid(pl)
        n = len(d)
        # loop exit: ratio <= R unless every document is Per-Doc
        mx, sm = pl.pass_ratios[-1]
        if strategy == P.STRATEGY_HYBRID:
            assert mx * N * 1_000_000 <= r_ppm * sm or len(pl.per_doc) == n
            assert len(pl.pass_ratios) == len(pl.per_doc) + 1
            # Per-Doc documents are the longest ones, popped in descending length
            lens = [d[k] for k in pl.per_doc]
            assert lens == sorted(lens, reverse=True)
            if pl.per_doc:
                assert min(lens) >= max([d[k] for k in range(n) if k not in pl.per_doc], default=0)
        elif strategy == P.STRATEGY_ALL_PER_DOC:
            assert len(pl.per_doc) == n
        else:
            assert len(pl.per_doc) == 0
        # determinism
        assert P.plan(d, N, r_ppm, strategy) == pl


def test_aligned_variant_invariants():
    """align = A > 1: still an exact cover with exactly C/N tokens per worker
    (Eq. 1, Eq. 2); A = 1 is Algorithm 1 itself; Per-Doc chunks start on the grid and have
    lengths that are multiples of A except the one ending its document; and on the bench recipes
    the cuts that are not on a multiple of 128 shrink to a handful."""
    for d, N, r_ppm, strategy in random_inputs(5, 300):
        assert P.plan(d, N, r_ppm, strategy, align=1) == P.plan(d, N, r_ppm, strategy)
        for A in (2, 4, 8, 16):
            pl = P.plan(d, N, r_ppm, strategy, align=A)
            check_valid(pl)
            assert P.plan(d, N, r_ppm, strategy, align=A) == pl
            if strategy == P.STRATEGY_ALL_PER_DOC:
                for k, x in enumerate(d):
                    q = x // (2 * N * A) * A
                    if q == 0:
                        continue
                    h = (x - 2 * N * q) // A * A
                    e = x - 2 * N * q - h
                    # the chunk grid h + c q is respected: chunks are never cut, so every cut
                    # of the document inside (h, d - e) is a grid point (the head item [0, h)
                    # and the ragged tail [d - e, d) are movable and may be cut anywhere)
                    cuts = {s.start for s in pl.shards if s.doc == k and h < s.start < x - e}
                    assert all((c - h) % q == 0 for c in cuts), (d, N, A, k, cuts)
    import fcp_inputs
    for name in ("8b", "longtail", "70b"):
        cfg = fcp_inputs.CONFIGS[name]
        for seed in (0, 1):
            d = fcp_inputs.doc_lengths(name, seed)
            off = [sum(1 for s in P.plan(d, cfg.N, align=A).shards if s.start % 128) for A in (1, 128)]
            assert off[1] <= cfg.N - 1 and off[1] <= off[0], (name, seed, off)
            check_valid(P.plan(d, cfg.N, align=128))


def test_per_doc_pair_identity_and_exact_balance():
    for N in (1, 2, 3, 4, 8):
        for q in (1, 2, 5):
            for r in (0, 1, 2 * N - 1):
                want = q * (2 * r + 2 * N * q + 1)
                for j in range(N):
                    got = brute_pairs(r + j * q, q) + brute_pairs(r + (2 * N - 1 - j) * q, q)
                    assert got == want
    # all documents multiples of 2N, all Per-Doc -> ratio exactly 1
    pl = P.plan([16, 32, 48, 8], 4, strategy=P.STRATEGY_ALL_PER_DOC)
    loads = P.rank_loads(pl)
    assert len(set(loads)) == 1 and P.imbalance_ppm(pl) == 1_000_000
    # chunks c and 2N-1-c on worker c
    pl = P.plan([16], 2, strategy=P.STRATEGY_ALL_PER_DOC)
    assert [(s.start, s.len, s.rank) for s in pl.shards] == [(0, 4, 0), (12, 4, 0), (4, 8, 1)]


def optimum_max_load(d, N):
    """Brute force over ALL token->worker assignments with C/N tokens each: a token at document
    position t costs t+1 pairs.  Lower bound for any sharding (Eq. 3)."""
    cost = [t + 1 for x in d for t in range(x)]
    C = len(cost)
    T = C // N
    best = None

    def rec(i, tok, load):
        nonlocal best
        if best is not None and max(load) >= best:
            return
        if i == C:
            best = max(load)
            return
        seen = set()
        for j in range(N):
            if tok[j] < T and (tok[j], load[j]) not in seen:
                seen.add((tok[j], load[j]))
                tok[j] += 1
                load[j] += cost[i]
                rec(i + 1, tok, load)
                tok[j] -= 1
                load[j] -= cost[i]
    rec(0, [0] * N, [0] * N)
    return best


def test_heuristic_never_beats_the_optimum():
    rng = np.random.default_rng(7)
    for _ in range(40):
        N = int(rng.integers(2, 4))
        n = int(rng.integers(1, 4))
        d = [int(x) for x in rng.integers(1, 6, size=n)]
        pad = (-sum(d)) % N
        if pad:
            d.append(pad)
        if sum(d) > 14:
            continue
        opt = optimum_max_load(d, N)
        for strategy in (0, 1, 2):
            pl = P.plan(d, N, 1_000_000, strategy)
            assert max(P.rank_loads(pl)) >= opt
        # with R = 1.0 the hybrid ends all-Per-Doc or exactly balanced
    assert optimum_max_load([2, 2], 2) == 3


def test_invalid_arguments():
    for bad in ([], [0, 4], [3, 4]):
        with pytest.raises(ValueError):
            P.plan(bad, 2)
    with pytest.raises(ValueError):
        P.plan([4, 4], 0)
    with pytest.raises(ValueError):
        P.plan([4, 4], 2, 999_999)


# ---------------------------------------------------------------------------------------------
# Per-Seq sharding (Llama3 CP baseline) — SURVEY 8(f) NEXT 3
# ---------------------------------------------------------------------------------------------
def test_per_seq_hand_worked_examples():
    """Worked by hand from PAPER.md:50 ("split into 2 x CP shards, each worker processes two
    shards"; chunks i and 2N-1-i as in PAPER.md:62).
    D=[8,8], N=2: chunks of 4 tokens -> rank0 {[0,4) of doc0, [4,8) of doc1}, rank1 {[4,8) of
    doc0, [0,4) of doc1}; W(0,4)=10, W(4,4)=26 -> loads 36/36.
    D=[12,4], N=2: rank0 {doc0[0,4), doc1[0,4)} = 10+10, rank1 {doc0[4,12)} (chunks 1 and 2 are
    contiguous and merge) = W(4,8) = 68 -> ratio 68*2/88 = 1.545 (the imbalance of Fig. 1(b))."""
    pl = P.plan([8, 8], 2, strategy=P.STRATEGY_PER_SEQ)
    assert pl.shards == (P.Shard(0, 0, 4, 0), P.Shard(1, 4, 4, 0), P.Shard(0, 4, 4, 1), P.Shard(1, 0, 4, 1))
    assert P.rank_loads(pl) == [36, 36] and pl.per_doc == ()
    pl = P.plan([12, 4], 2, strategy=P.STRATEGY_PER_SEQ)
    assert pl.shards == (P.Shard(0, 0, 4, 0), P.Shard(1, 0, 4, 0), P.Shard(0, 4, 8, 1))
    assert P.rank_loads(pl) == [20, 68]
    assert P.imbalance_ppm(pl) == 68 * 2 * 1_000_000 // 88
    with pytest.raises(ValueError):
        P.plan([10, 4], 2, strategy=P.STRATEGY_PER_SEQ)      # C = 14 is not a multiple of 2N = 4


def test_per_seq_invariants_and_single_document_equals_per_doc():
    rng = np.random.default_rng(12)
    for _ in range(60):
        N = int(rng.integers(1, 6))
        n = int(rng.integers(1, 7))
        d = [int(x) for x in rng.integers(1, 40, size=n)]
        pad = (-sum(d)) % (2 * N)
        d[-1] += pad
        pl = P.plan(d, N, strategy=P.STRATEGY_PER_SEQ)
        C = sum(d)
        # Eq. 1: every token of every document exactly once; Eq. 2: C/N tokens per worker
        seen = [np.zeros(x, dtype=int) for x in d]
        for s in pl.shards:
            seen[s.doc][s.start:s.start + s.len] += 1
        assert all((v == 1).all() for v in seen)
        assert P.rank_tokens(pl) == [C // N] * N
        assert sum(P.rank_loads(pl)) == sum(x * (x + 1) // 2 for x in d)
        # chunk structure: worker j holds global tokens of chunks j and 2N-1-j only
        q = C // (2 * N)
        off = np.concatenate([[0], np.cumsum(d)])
        for s in pl.shards:
            g0, g1 = off[s.doc] + s.start, off[s.doc] + s.start + s.len - 1
            for g in (g0, g1):
                c = g // q
                assert s.rank == (c if c < N else 2 * N - 1 - c)
    # one document: Per-Seq is exactly all-Per-Doc when 2N divides it
    for N in (1, 2, 4):
        a = P.plan([16 * N], N, strategy=P.STRATEGY_PER_SEQ)
        b = P.plan([16 * N], N, strategy=P.STRATEGY_ALL_PER_DOC)
        assert a.shards == b.shards
