"""Oracle: document-masked causal attention, forward and backward, and the partial-result
merge (TEST INFRASTRUCTURE, see oracle/__init__.py).  numpy fp64 throughout.

Definition ("intra-document causal masking"; "the Q tensor of each
token only computes attention with the prefix part of the KV tensor"): for every document k
separately and every query head h (kv head h // G, G = Hq/Hkv)

    S = scale * Q_k K_k^T,  S[t, j] = -inf for j > t,  P = softmax_rows(S),  O = P V_k,
    lse[t] = log sum_j exp S[t, j]                       (natural log, on scaled scores)

Backward for upstream dO (the paper only states that K/V are needed again and gradients are
synchronised; the formulas are the derivative of the definition above):

    dV = P^T dO,  dP = dO V^T,  delta = rowsum(dO o O),  dS = P o (dP - delta),
    dQ = scale * dS K,  dK = scale * dS^T Q;    dK, dV of a kv head sum over its G query heads.

Layouts: q, o, dO, dq [rows, Hq, D];  k, v, dk, dv [rows, Hkv, D];  lse [Hq, rows].

`packed_*` is the plain per-document definition.  `shard_*` is what one CP worker computes
for one shard (doc k, prefix p, length s): query rows [p, p+s) of the document against keys
[0, p+s), row t seeing keys 0..p+t.  The two are separate code so that agreement between them
("plan invariance") is a real check.  Work is row-blocked only so a 78K-token document does not
need a 49 GB score matrix; there is no online softmax and no tiling of the key axis.
"""

import numpy as np

ROW_BLOCK = 256


def _group(Hq, Hkv):
    if Hq % Hkv:
        raise ValueError("Hq must be a multiple of Hkv")
    return Hq // Hkv


# --------------------------------------------------------------------------------------
# plain per-document definition
# --------------------------------------------------------------------------------------

def doc_fwd(q, k, v, scale):
    """One whole document.  q [d,Hq,D], k,v [d,Hkv,D] -> o [d,Hq,D], lse [Hq,d]."""
    d, Hq, D = q.shape
    Hkv = k.shape[1]
    G = _group(Hq, Hkv)
    o = np.zeros((d, Hq, D))
    lse = np.zeros((Hq, d))
    for h in range(Hq):
        kh, vh = k[:, h // G, :], v[:, h // G, :]
        for t0 in range(0, d, ROW_BLOCK):
            t1 = min(d, t0 + ROW_BLOCK)
            S = scale * (q[t0:t1, h, :] @ kh[:t1].T)                     # [B, t1]
            t = np.arange(t0, t1)[:, None]
            j = np.arange(t1)[None, :]
            S = np.where(j > t, -np.inf, S)
            m = S.max(axis=1, keepdims=True)
            e = np.exp(S - m)
            z = e.sum(axis=1, keepdims=True)
            o[t0:t1, h, :] = (e / z) @ vh[:t1]
            lse[h, t0:t1] = (m + np.log(z))[:, 0]
    return o, lse


def doc_bwd(q, k, v, do, scale):
    """One whole document.  Returns dq [d,Hq,D], dk, dv [d,Hkv,D]."""
    d, Hq, D = q.shape
    Hkv = k.shape[1]
    G = _group(Hq, Hkv)
    o, lse = doc_fwd(q, k, v, scale)
    dq = np.zeros_like(q)
    dk = np.zeros_like(k)
    dv = np.zeros_like(v)
    for h in range(Hq):
        g = h // G
        kh, vh = k[:, g, :], v[:, g, :]
        for t0 in range(0, d, ROW_BLOCK):
            t1 = min(d, t0 + ROW_BLOCK)
            S = scale * (q[t0:t1, h, :] @ kh[:t1].T)
            t = np.arange(t0, t1)[:, None]
            j = np.arange(t1)[None, :]
            P = np.where(j > t, 0.0, np.exp(S - lse[h, t0:t1, None]))
            dO = do[t0:t1, h, :]
            dv[:t1, g, :] += P.T @ dO
            dP = dO @ vh[:t1].T
            delta = (dO * o[t0:t1, h, :]).sum(axis=1, keepdims=True)
            dS = P * (dP - delta)
            dq[t0:t1, h, :] = scale * (dS @ kh[:t1])
            dk[:t1, g, :] += scale * (dS.T @ q[t0:t1, h, :])
    return dq, dk, dv


def packed_fwd(Q, K, V, d, scale):
    """Packed sequence of documents with lengths d.  Global token order."""
    o = np.zeros_like(Q)
    lse = np.zeros((Q.shape[1], Q.shape[0]))
    off = 0
    for dk_ in d:
        o[off:off + dk_], lse[:, off:off + dk_] = doc_fwd(Q[off:off + dk_], K[off:off + dk_],
                                                          V[off:off + dk_], scale)
        off += dk_
    return o, lse


def packed_bwd(Q, K, V, dO, d, scale):
    dQ, dK, dV = np.zeros_like(Q), np.zeros_like(K), np.zeros_like(V)
    off = 0
    for dk_ in d:
        sl = slice(off, off + dk_)
        dQ[sl], dK[sl], dV[sl] = doc_bwd(Q[sl], K[sl], V[sl], dO[sl], scale)
        off += dk_
    return dQ, dK, dV


# --------------------------------------------------------------------------------------
# what one CP worker computes for one shard
# --------------------------------------------------------------------------------------

def _visible(p, t0, t1, L, kv_len):
    """Boolean [t1-t0, L]: key j visible to shard row t iff j <= p + t and j < kv_len."""
    t = np.arange(t0, t1)[:, None]
    j = np.arange(L)[None, :]
    return (j <= p + t) & (j < kv_len)


def shard_fwd(q, k, v, p, scale, kv_len=None):
    """Shard rows q [s,Hq,D] at document positions p..p+s-1 against keys k,v [L,Hkv,D]
    (document positions 0..L-1; with a KV *piece* p may be negative).
    Row t sees keys j <= p+t, j < kv_len (default L).  Rows that see no key give o = 0,
    lse = -inf.  Returns o [s,Hq,D], lse [Hq,s]."""
    s, Hq, D = q.shape
    L, Hkv = k.shape[0], k.shape[1]
    kv_len = L if kv_len is None else kv_len
    G = _group(Hq, Hkv)
    o = np.zeros((s, Hq, D))
    lse = np.full((Hq, s), -np.inf)
    for h in range(Hq):
        kh, vh = k[:, h // G, :], v[:, h // G, :]
        for t0 in range(0, s, ROW_BLOCK):
            t1 = min(s, t0 + ROW_BLOCK)
            Lb = max(0, min(kv_len, p + t1))            # no row of the block sees beyond this
            if Lb == 0:
                continue
            vis = _visible(p, t0, t1, Lb, kv_len)
            S = np.where(vis, scale * (q[t0:t1, h, :] @ kh[:Lb].T), -np.inf)
            m = S.max(axis=1, keepdims=True)
            any_vis = np.isfinite(m)
            m = np.where(any_vis, m, 0.0)
            e = np.exp(S - m)
            z = e.sum(axis=1, keepdims=True)
            with np.errstate(divide="ignore", invalid="ignore"):
                o[t0:t1, h, :] = np.where(any_vis, (e / np.where(any_vis, z, 1.0)) @ vh[:Lb], 0.0)
                lse[h, t0:t1] = np.where(any_vis, m + np.log(np.where(any_vis, z, 1.0)),
                                         -np.inf)[:, 0]
    return o, lse


def shard_bwd(q, k, v, o, lse, do, p, scale, kv_len=None):
    """Backward of shard_fwd.  `o`, `lse` are the FINAL (merged, if the keys were processed in
    pieces) output and log-sum-exp of the rows ("backward through pieces").
    Returns dq [s,Hq,D] and this shard's contribution dk, dv [L,Hkv,D]."""
    s, Hq, D = q.shape
    L, Hkv = k.shape[0], k.shape[1]
    kv_len = L if kv_len is None else kv_len
    G = _group(Hq, Hkv)
    dq = np.zeros((s, Hq, D))
    dk = np.zeros((L, Hkv, D))
    dv = np.zeros((L, Hkv, D))
    for h in range(Hq):
        g = h // G
        kh, vh = k[:, g, :], v[:, g, :]
        for t0 in range(0, s, ROW_BLOCK):
            t1 = min(s, t0 + ROW_BLOCK)
            Lb = max(0, min(kv_len, p + t1))
            if Lb == 0:
                continue
            vis = _visible(p, t0, t1, Lb, kv_len)
            S = scale * (q[t0:t1, h, :] @ kh[:Lb].T)
            row_lse = lse[h, t0:t1, None]
            with np.errstate(invalid="ignore", over="ignore"):
                P = np.where(vis & np.isfinite(row_lse), np.exp(S - row_lse), 0.0)
            dO = do[t0:t1, h, :]
            dv[:Lb, g, :] += P.T @ dO
            dP = dO @ vh[:Lb].T
            delta = (dO * o[t0:t1, h, :]).sum(axis=1, keepdims=True)
            dS = P * (dP - delta)
            dq[t0:t1, h, :] = scale * (dS @ kh[:Lb])
            dk[:Lb, g, :] += scale * (dS.T @ q[t0:t1, h, :])
    return dq, dk, dv


def shard_rows_fwd(q_rows, k, v, key_counts, scale):
    """Row-at-a-time forward for sampled rows (used for parity at sizes where the full oracle
    is too slow).  q_rows [m,Hq,D]; row i sees keys 0..key_counts[i]-1 of k,v [L,Hkv,D]."""
    m, Hq, D = q_rows.shape
    G = _group(Hq, k.shape[1])
    o = np.zeros((m, Hq, D))
    lse = np.zeros((Hq, m))
    for i in range(m):
        n = int(key_counts[i])
        for h in range(Hq):
            sc = scale * (k[:n, h // G, :] @ q_rows[i, h, :])
            mx = sc.max()
            e = np.exp(sc - mx)
            z = e.sum()
            o[i, h, :] = (e / z) @ v[:n, h // G, :]
            lse[h, i] = mx + np.log(z)
    return o, lse


def shard_rows_bwd_dq(q_rows, k, v, do_rows, key_counts, scale):
    """Row-at-a-time dq for sampled rows (parity at sizes where the full oracle is too slow):
    dq of a query row depends on that row alone.  For row i with n = key_counts[i] visible keys
    p = softmax(scale q.K[:n]), o = p V[:n], delta = dO.o, dp = V[:n] dO,
    ds = p o (dp - delta), dq = scale ds K[:n]  (the formulas at the top of this file).
    q_rows, do_rows [m,Hq,D]; k,v [L,Hkv,D] -> dq [m,Hq,D]."""
    m, Hq, D = q_rows.shape
    G = _group(Hq, k.shape[1])
    dq = np.zeros((m, Hq, D))
    for i in range(m):
        n = int(key_counts[i])
        for h in range(Hq):
            kh, vh = k[:n, h // G, :], v[:n, h // G, :]
            sc = scale * (kh @ q_rows[i, h, :])
            e = np.exp(sc - sc.max())
            p = e / e.sum()
            o = p @ vh
            delta = float(do_rows[i, h, :] @ o)
            dp = vh @ do_rows[i, h, :]
            ds = p * (dp - delta)
            dq[i, h, :] = scale * (ds @ kh)
    return dq


# --------------------------------------------------------------------------------------
# partial-result aggregation
# --------------------------------------------------------------------------------------

def merge(o_a, lse_a, o_b, lse_b):
    """Combine attention partials over two disjoint key sets.
    lse = log(e^lse_a + e^lse_b), o = e^(lse_a-lse) o_a + e^(lse_b-lse) o_b.
    o_* [rows,H,D], lse_* [H,rows].  A partial with lse = -inf has weight 0."""
    m = np.maximum(lse_a, lse_b)
    m_safe = np.where(np.isfinite(m), m, 0.0)
    ea = np.exp(lse_a - m_safe)
    eb = np.exp(lse_b - m_safe)
    z = ea + eb
    with np.errstate(divide="ignore", invalid="ignore"):
        lse = np.where(z > 0, m_safe + np.log(np.where(z > 0, z, 1.0)), -np.inf)
        wa = np.where(z > 0, ea / np.where(z > 0, z, 1.0), 0.0)
        wb = np.where(z > 0, eb / np.where(z > 0, z, 1.0), 0.0)
    o = wa.T[:, :, None] * o_a + wb.T[:, :, None] * o_b
    return o, lse


# --------------------------------------------------------------------------------------
# one CP worker: all of its shards, in the rank-local layouts of the C-ABI
# --------------------------------------------------------------------------------------

def rank_fwd(q_local, k_gath, v_gath, cu_seqlens_q, q_pos_off, shard_seg, cu_seqlens_k, scale):
    """q_local [n_q,Hq,D] rank-local rows; k_gath,v_gath [n_kv,Hkv,D] gathered KV.
    Returns o [n_q,Hq,D], lse [Hq,n_q]."""
    n_q, Hq, D = q_local.shape
    o = np.zeros((n_q, Hq, D))
    lse = np.zeros((Hq, n_q))
    for i in range(len(q_pos_off)):
        a, b = int(cu_seqlens_q[i]), int(cu_seqlens_q[i + 1])
        g = int(shard_seg[i])
        ka, kb = int(cu_seqlens_k[g]), int(cu_seqlens_k[g + 1])
        o[a:b], lse[:, a:b] = shard_fwd(q_local[a:b], k_gath[ka:kb], v_gath[ka:kb],
                                        int(q_pos_off[i]), scale)
    return o, lse


def rank_bwd(q_local, k_gath, v_gath, o, lse, do, cu_seqlens_q, q_pos_off, shard_seg,
             cu_seqlens_k, scale):
    """Returns dq [n_q,Hq,D] and dk, dv [n_kv,Hkv,D] in gathered-KV order, holding only this
    rank's queries' contributions (global dK = sum over ranks of scatter-add)."""
    dq = np.zeros_like(q_local)
    dk = np.zeros_like(k_gath)
    dv = np.zeros_like(v_gath)
    for i in range(len(q_pos_off)):
        a, b = int(cu_seqlens_q[i]), int(cu_seqlens_q[i + 1])
        g = int(shard_seg[i])
        ka, kb = int(cu_seqlens_k[g]), int(cu_seqlens_k[g + 1])
        dq[a:b], dk_i, dv_i = shard_bwd(q_local[a:b], k_gath[ka:kb], v_gath[ka:kb], o[a:b],
                                        lse[:, a:b], do[a:b], int(q_pos_off[i]), scale)
        dk[ka:kb] += dk_i
        dv[ka:kb] += dv_i
    return dq, dk, dv
