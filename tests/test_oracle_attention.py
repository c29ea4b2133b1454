"""Pins for oracle/attention.py: brute force, library special case, closed forms, plan
invariance, merge identity, finite differences, GQA (SURVEY.md section 8(c1) pins 1-8)."""
import math

import numpy as np
import pytest

from oracle import attention as A
from oracle import planner as P
from oracle import kvselect as KV


def rnd(rng, *shape):
    return rng.standard_normal(shape)


def brute_doc(q, k, v, scale):
    """Explicit loops over (t, j <= t): the definition at PAPER.md:46 with nothing else."""
    d, Hq, D = q.shape
    G = Hq // k.shape[1]
    o = np.zeros_like(q)
    lse = np.zeros((Hq, d))
    for h in range(Hq):
        for t in range(d):
            sc = [scale * sum(q[t, h, c] * k[j, h // G, c] for c in range(D)) for j in range(t + 1)]
            z = sum(math.exp(x) for x in sc)
            lse[h, t] = math.log(z)
            for j in range(t + 1):
                w = math.exp(sc[j]) / z
                for c in range(D):
                    o[t, h, c] += w * v[j, h // G, c]
    return o, lse


def test_bruteforce_tiny():
    rng = np.random.default_rng(0)
    for d, Hq, Hkv, D in [(1, 1, 1, 2), (5, 2, 1, 3), (16, 4, 2, 4)]:
        q, k, v = rnd(rng, d, Hq, D), rnd(rng, d, Hkv, D), rnd(rng, d, Hkv, D)
        o, lse = A.doc_fwd(q, k, v, 0.7)
        bo, bl = brute_doc(q, k, v, 0.7)
        np.testing.assert_allclose(o, bo, rtol=0, atol=1e-12)
        np.testing.assert_allclose(lse, bl, rtol=0, atol=1e-12)
        # shard form with p = 0 on the whole document is the same thing
        so, sl = A.shard_fwd(q, k, v, 0, 0.7)
        np.testing.assert_allclose(so, bo, atol=1e-12)
        np.testing.assert_allclose(sl, bl, atol=1e-12)
        # a shard in the middle of the document
        for p, s in [(0, d), (d // 2, d - d // 2), (d - 1, 1)]:
            so, sl = A.shard_fwd(q[p:p + s], k, v, p, 0.7)
            np.testing.assert_allclose(so, bo[p:p + s], atol=1e-12)
            np.testing.assert_allclose(sl, bl[:, p:p + s], atol=1e-12)


def test_library_special_case_sdpa():
    torch = pytest.importorskip("torch")
    rng = np.random.default_rng(1)
    d, Hq, Hkv, D = 300, 4, 2, 16          # spans the oracle's row blocks
    scale = 1.0 / math.sqrt(D)
    q, k, v, do = rnd(rng, d, Hq, D), rnd(rng, d, Hkv, D), rnd(rng, d, Hkv, D), rnd(rng, d, Hq, D)
    tq = torch.tensor(q, requires_grad=True)
    tk = torch.tensor(k, requires_grad=True)
    tv = torch.tensor(v, requires_grad=True)
    G = Hq // Hkv
    out = torch.nn.functional.scaled_dot_product_attention(
        tq.permute(1, 0, 2)[None], tk.permute(1, 0, 2).repeat_interleave(G, 0)[None],
        tv.permute(1, 0, 2).repeat_interleave(G, 0)[None], is_causal=True, scale=scale)
    out = out[0].permute(1, 0, 2)
    out.backward(torch.tensor(do))
    o, lse = A.doc_fwd(q, k, v, scale)
    np.testing.assert_allclose(o, out.detach().numpy(), atol=1e-11)
    dq, dk, dv = A.doc_bwd(q, k, v, do, scale)
    np.testing.assert_allclose(dq, tq.grad.numpy(), atol=1e-10)
    np.testing.assert_allclose(dk, tk.grad.numpy(), atol=1e-10)
    np.testing.assert_allclose(dv, tv.grad.numpy(), atol=1e-10)
    # shard form, backward
    so, sl = A.shard_fwd(q, k, v, 0, scale)
    sdq, sdk, sdv = A.shard_bwd(q, k, v, so, sl, do, 0, scale)
    np.testing.assert_allclose(sdq, tq.grad.numpy(), atol=1e-10)
    np.testing.assert_allclose(sdk, tk.grad.numpy(), atol=1e-10)
    np.testing.assert_allclose(sdv, tv.grad.numpy(), atol=1e-10)


def test_closed_forms():
    rng = np.random.default_rng(2)
    s, p, H, D = 37, 11, 2, 4
    L = p + s
    q, v, do = rnd(rng, s, H, D), rnd(rng, L, H, D), rnd(rng, s, H, D)
    k0 = np.zeros((L, H, D))
    o, lse = A.shard_fwd(q, k0, v, p, 0.5)
    t = np.arange(s)
    # K = 0: lse encodes exactly the number of visible keys; o is the running mean of V
    np.testing.assert_allclose(lse, np.broadcast_to(np.log(p + t + 1.0), (H, s)), atol=1e-13)
    csum = np.cumsum(v, axis=0)
    np.testing.assert_allclose(o, csum[p:p + s] / (p + t + 1.0)[:, None, None], atol=1e-12)
    dq, dk, dv = A.shard_bwd(q, k0, v, o, lse, do, p, 0.5)
    want_dv = np.zeros_like(v)
    for j in range(L):
        for tt in range(s):
            if j <= p + tt:
                want_dv[j] += do[tt] / (p + tt + 1.0)
    np.testing.assert_allclose(dv, want_dv, atol=1e-12)
    np.testing.assert_allclose(dq, 0, atol=1e-12)          # K = 0 -> dQ = scale dS K = 0
    # first token of a document: o_0 = v_0, lse_0 = scale q_0.k_0
    k = rnd(rng, L, H, D)
    o, lse = A.doc_fwd(q[:5], k[:5], v[:5], 0.5)
    np.testing.assert_allclose(o[0], v[0], atol=1e-13)
    np.testing.assert_allclose(lse[:, 0], 0.5 * (q[0] * k[0]).sum(-1), atol=1e-13)
    # all V rows equal -> o = v*, dQ = dK = 0
    vstar = np.broadcast_to(rnd(rng, 1, H, D), (L, H, D)).copy()
    o, lse = A.shard_fwd(q, k, vstar, p, 0.5)
    np.testing.assert_allclose(o, np.broadcast_to(vstar[:1], o.shape), atol=1e-12)
    dq, dk, dv = A.shard_bwd(q, k, vstar, o, lse, do, p, 0.5)
    np.testing.assert_allclose(dq, 0, atol=1e-12)
    np.testing.assert_allclose(dk, 0, atol=1e-12)
    # bounds: |o| <= max |v| over visible rows
    o, lse = A.shard_fwd(q, k, v, p, 0.5)
    assert np.abs(o).max() <= np.abs(v).max() + 1e-12


def test_finite_differences():
    rng = np.random.default_rng(3)
    d, Hq, Hkv, D, scale = 8, 2, 1, 4, 0.6
    q, k, v, do = rnd(rng, d, Hq, D), rnd(rng, d, Hkv, D), rnd(rng, d, Hkv, D), rnd(rng, d, Hq, D)
    dq, dk, dv = A.doc_bwd(q, k, v, do, scale)

    def f(q_, k_, v_):
        return (A.doc_fwd(q_, k_, v_, scale)[0] * do).sum()
    h = 1e-5
    for arr, grad, which in ((q, dq, 0), (k, dk, 1), (v, dv, 2)):
        num = np.zeros_like(arr)
        it = np.nditer(arr, flags=["multi_index"])
        for _ in it:
            i = it.multi_index
            args = [q.copy(), k.copy(), v.copy()]
            args[which][i] += h
            fp = f(*args)
            args[which][i] -= 2 * h
            fm = f(*args)
            num[i] = (fp - fm) / (2 * h)
        np.testing.assert_allclose(grad, num, atol=2e-8)


def test_gqa_equals_repeated_mha():
    rng = np.random.default_rng(4)
    d, Hq, Hkv, D, scale = 40, 6, 2, 8, 0.3
    G = Hq // Hkv
    q, k, v, do = rnd(rng, d, Hq, D), rnd(rng, d, Hkv, D), rnd(rng, d, Hkv, D), rnd(rng, d, Hq, D)
    kr, vr = np.repeat(k, G, axis=1), np.repeat(v, G, axis=1)
    o, lse = A.doc_fwd(q, k, v, scale)
    o2, lse2 = A.doc_fwd(q, kr, vr, scale)
    np.testing.assert_allclose(o, o2, atol=1e-13)
    np.testing.assert_allclose(lse, lse2, atol=1e-13)
    dq, dk, dv = A.doc_bwd(q, k, v, do, scale)
    dq2, dk2, dv2 = A.doc_bwd(q, kr, vr, do, scale)
    np.testing.assert_allclose(dq, dq2, atol=1e-12)
    np.testing.assert_allclose(dk, dk2.reshape(d, Hkv, G, D).sum(2), atol=1e-12)
    np.testing.assert_allclose(dv, dv2.reshape(d, Hkv, G, D).sum(2), atol=1e-12)


def run_plan(pl, Q, K, V, dO, scale):
    """Every rank's results put back into global order; dK,dV scatter-added."""
    C = Q.shape[0]
    o = np.zeros_like(Q)
    lse = np.zeros((Q.shape[1], C))
    dq = np.zeros_like(Q)
    dk = np.zeros_like(K)
    dv = np.zeros_like(V)
    for r in range(pl.n_ranks):
        lay = KV.rank_layout(pl, r)
        qi = KV.q_token_index(pl, r)
        gi = KV.gather_index(pl, r)
        args = (lay.cu_seqlens_q, lay.q_pos_off, lay.shard_seg, lay.cu_seqlens_k, scale)
        o_r, lse_r = A.rank_fwd(Q[qi], K[gi], V[gi], *args)
        dq_r, dk_r, dv_r = A.rank_bwd(Q[qi], K[gi], V[gi], o_r, lse_r, dO[qi], *args)
        o[qi], lse[:, qi], dq[qi] = o_r, lse_r, dq_r
        np.add.at(dk, gi, dk_r)
        np.add.at(dv, gi, dv_r)
    return o, lse, dq, dk, dv


def test_plan_invariance():
    rng = np.random.default_rng(5)
    Hq, Hkv, D, scale = 4, 2, 8, 0.35
    for trial in range(12):
        N = int(rng.integers(1, 5))
        d = [int(x) for x in rng.integers(1, 90, size=int(rng.integers(1, 7)))]
        pad = (-sum(d)) % N
        if pad:
            d.append(pad)
        C = sum(d)
        Q, K, V, dO = rnd(rng, C, Hq, D), rnd(rng, C, Hkv, D), rnd(rng, C, Hkv, D), rnd(rng, C, Hq, D)
        want_o, want_lse = A.packed_fwd(Q, K, V, d, scale)
        want = (want_o, want_lse) + A.packed_bwd(Q, K, V, dO, d, scale)
        for strategy in (0, 1, 2):
            pl = P.plan(d, N, 1_050_000, strategy)
            got = run_plan(pl, Q, K, V, dO, scale)
            for g, w in zip(got, want):
                np.testing.assert_allclose(g, w, atol=1e-11)


def test_merge_identity():
    rng = np.random.default_rng(6)
    s, p, Hq, Hkv, D, scale = 50, 30, 4, 2, 8, 0.4
    L = p + s
    q, k, v = rnd(rng, s, Hq, D), rnd(rng, L, Hkv, D), rnd(rng, L, Hkv, D)
    o, lse = A.shard_fwd(q, k, v, p, scale)
    for c in (1, 17, 30, 45, 79):
        oa, la = A.shard_fwd(q, k[:c], v[:c], p, scale)              # keys [0, c)
        ob, lb = A.shard_fwd(q, k[c:], v[c:], p - c, scale)          # keys [c, L)
        om, lm = A.merge(oa, la, ob, lb)
        np.testing.assert_allclose(om, o, atol=1e-12)
        np.testing.assert_allclose(lm, lse, atol=1e-12)
        om2, lm2 = A.merge(ob, lb, oa, la)                           # commutative
        np.testing.assert_allclose(om2, om, atol=1e-13)
        if c > p:                                                    # some rows see nothing in B
            assert np.isneginf(lb[:, :c - p]).all() and (ob[:c - p] == 0).all()
    # three pieces, both association orders
    c1, c2 = 20, 55
    parts = [A.shard_fwd(q, k[:c1], v[:c1], p, scale),
             A.shard_fwd(q, k[c1:c2], v[c1:c2], p - c1, scale),
             A.shard_fwd(q, k[c2:], v[c2:], p - c2, scale)]
    left = A.merge(*A.merge(*parts[0], *parts[1]), *parts[2])
    right = A.merge(*parts[0], *A.merge(*parts[1], *parts[2]))
    np.testing.assert_allclose(left[0], o, atol=1e-12)
    np.testing.assert_allclose(right[0], o, atol=1e-12)
    np.testing.assert_allclose(left[1], right[1], atol=1e-12)
    # backward through pieces: each piece uses the merged lse / o; dq adds, dk/dv concatenate
    do = rnd(rng, s, Hq, D)
    dq, dk, dv = A.shard_bwd(q, k, v, o, lse, do, p, scale)
    c = 45
    dqa, dka, dva = A.shard_bwd(q, k[:c], v[:c], o, lse, do, p, scale)
    dqb, dkb, dvb = A.shard_bwd(q, k[c:], v[c:], o, lse, do, p - c, scale)
    np.testing.assert_allclose(dqa + dqb, dq, atol=1e-12)
    np.testing.assert_allclose(np.concatenate([dka, dkb]), dk, atol=1e-12)
    np.testing.assert_allclose(np.concatenate([dva, dvb]), dv, atol=1e-12)
    # kv_len restriction == truncating the arrays
    o1, l1 = A.shard_fwd(q, k, v, p, scale, kv_len=c)
    np.testing.assert_allclose(o1, oa_ := A.shard_fwd(q, k[:c], v[:c], p, scale)[0], atol=1e-13)


def test_sampled_rows_match_full():
    rng = np.random.default_rng(8)
    s, p, Hq, Hkv, D, scale = 20, 13, 4, 2, 8, 0.4
    q, k, v = rnd(rng, s, Hq, D), rnd(rng, p + s, Hkv, D), rnd(rng, p + s, Hkv, D)
    o, lse = A.shard_fwd(q, k, v, p, scale)
    rows = np.array([0, 7, 19])
    so, sl = A.shard_rows_fwd(q[rows], k, v, p + rows + 1, scale)
    np.testing.assert_allclose(so, o[rows], atol=1e-13)
    np.testing.assert_allclose(sl, lse[:, rows], atol=1e-13)
    # sampled dq rows: equal to the full backward (itself pinned by SDPA autograd and central
    # differences) on the same rows, and to a central difference of the row's own loss
    do = rnd(rng, s, Hq, D)
    dq, _, _ = A.shard_bwd(q, k, v, o, lse, do, p, scale)
    sdq = A.shard_rows_bwd_dq(q[rows], k, v, do[rows], p + rows + 1, scale)
    np.testing.assert_allclose(sdq, dq[rows], atol=1e-13)
    i, h, c, eps = 1, 2, 3, 1e-6
    def loss(qq):
        oo, _ = A.shard_rows_fwd(qq, k, v, p + rows + 1, scale)
        return float((oo * do[rows]).sum())
    qp, qm = q[rows].copy(), q[rows].copy()
    qp[i, h, c] += eps
    qm[i, h, c] -= eps
    assert abs((loss(qp) - loss(qm)) / (2 * eps) - sdq[i, h, c]) < 1e-7


def test_local_prefix_split_merges_to_the_packed_result():
    """attention over the LOCAL and the PREFIX piece of every rank, merged
    (PAPER.md:64, 234), equals the plain packed definition — forward and, with the
    merged o / lse, backward (dq adds over the pieces, dK / dV scatter-add)."""
    rng = np.random.default_rng(15)
    Hq, Hkv, D, scale = 4, 2, 8, 0.3
    for trial in range(6):
        N = int(rng.integers(1, 5))
        d = [int(x) for x in rng.integers(1, 70, size=int(rng.integers(1, 6)))]
        pad = (-sum(d)) % N
        if pad:
            d.append(pad)
        C = sum(d)
        Q, K, V, dO = rnd(rng, C, Hq, D), rnd(rng, C, Hkv, D), rnd(rng, C, Hkv, D), rnd(rng, C, Hq, D)
        want_o, want_lse = A.packed_fwd(Q, K, V, d, scale)
        want_dq, want_dk, want_dv = A.packed_bwd(Q, K, V, dO, d, scale)
        for strategy in (0, 1):
            pl = P.plan(d, N, 1_050_000, strategy)
            o, lse = np.zeros_like(Q), np.zeros((Hq, C))
            dq, dk, dv = np.zeros_like(Q), np.zeros_like(K), np.zeros_like(V)
            for r in range(N):
                qi = KV.q_token_index(pl, r)
                part = {}
                for piece in (KV.PIECE_LOCAL, KV.PIECE_PREFIX):
                    L = KV.piece_layout(pl, r, piece)
                    gi = KV.piece_gather_index(pl, r, piece)
                    part[piece] = (L, gi) + A.rank_fwd(Q[qi], K[gi], V[gi], L.cu_seqlens_q,
                                                       L.q_pos_off, L.shard_seg, L.cu_seqlens_k, scale)
                o_r, lse_r = A.merge(*part[KV.PIECE_LOCAL][2:], *part[KV.PIECE_PREFIX][2:])
                o[qi], lse[:, qi] = o_r, lse_r
                for piece in (KV.PIECE_LOCAL, KV.PIECE_PREFIX):
                    L, gi = part[piece][:2]
                    dq_p, dk_p, dv_p = A.rank_bwd(Q[qi], K[gi], V[gi], o_r, lse_r, dO[qi],
                                                  L.cu_seqlens_q, L.q_pos_off, L.shard_seg,
                                                  L.cu_seqlens_k, scale)
                    dq[qi] += dq_p
                    np.add.at(dk, gi, dk_p)
                    np.add.at(dv, gi, dv_p)
            for g, w in zip((o, lse, dq, dk, dv), (want_o, want_lse, want_dq, want_dk, want_dv)):
                np.testing.assert_allclose(g, w, atol=1e-11)


def _arbitrary_plans():
    """hypothesis strategy: ANY exact cover of the documents by shards with ANY rank assignment
    (not the planner's output, not token-balanced) — SURVEY 8(c1) pin 4."""
    from hypothesis import strategies as st

    @st.composite
    def build(draw):
        n = draw(st.integers(1, 4))
        d = [draw(st.integers(1, 24)) for _ in range(n)]
        N = draw(st.integers(1, 4))
        shards = []
        for k, dk in enumerate(d):
            cuts = sorted(set(draw(st.lists(st.integers(1, dk), max_size=4)) + [dk]))
            a = 0
            for b in cuts:
                if b > a:
                    shards.append(P.Shard(k, a, b - a, draw(st.integers(0, N - 1))))
                    a = b
        shards.sort(key=lambda s: (s.rank, s.doc, s.start))
        merged = []                      # canonical form: contiguous neighbours on a rank merged
        for s in shards:
            m = merged[-1] if merged else None
            if m and (m.rank, m.doc) == (s.rank, s.doc) and m.start + m.len == s.start:
                merged[-1] = P.Shard(m.doc, m.start, m.len + s.len, m.rank)
            else:
                merged.append(s)
        return P.Plan(tuple(d), N, tuple(merged), (), ())
    return build()


def test_plan_invariance_for_arbitrary_valid_plans():
    from hypothesis import given, settings, HealthCheck

    @settings(max_examples=40, deadline=None, derandomize=True,
              suppress_health_check=list(HealthCheck))
    @given(_arbitrary_plans())
    def check(pl):
        rng = np.random.default_rng(len(pl.shards) * 1000 + sum(pl.d))
        Hq, Hkv, D, scale = 2, 1, 4, 0.45
        C = sum(pl.d)
        Q, K, V, dO = rnd(rng, C, Hq, D), rnd(rng, C, Hkv, D), rnd(rng, C, Hkv, D), rnd(rng, C, Hq, D)
        want_o, want_lse = A.packed_fwd(Q, K, V, list(pl.d), scale)
        want = (want_o, want_lse) + A.packed_bwd(Q, K, V, dO, list(pl.d), scale)
        for g, w in zip(run_plan(pl, Q, K, V, dO, scale), want):
            np.testing.assert_allclose(g, w, atol=1e-11)
        # and the gather list of every rank is exactly what its rows need
        for r in range(pl.n_ranks):
            need = set()
            off = KV.doc_offsets(pl.d)
            for s in pl.shards:
                if s.rank == r:
                    need.update(range(off[s.doc], off[s.doc] + s.start + s.len))
            assert sorted(need) == list(KV.gather_index(pl, r))
    check()
