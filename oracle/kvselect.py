"""Oracle: sharding-aware KV selection (TEST INFRASTRUCTURE, see oracle/__init__.py).

PAPER.md section 3.2: a document held whole by one worker needs no KV
exchange; a sharded document needs, on each worker, the prefix up to that worker's longest
shard end ("the Q tensor of each token only computes attention with the prefix part of the KV
tensor"); the prefixes are compacted into one contiguous buffer.

Definitions:
  off_k    = sum_{k'<k} d_k'                         global token offset of document k
  E_r(k)   = max{p+s : shard (k,p,s) on rank r}      0 if rank r holds no query of document k
  gather list of r = for k ascending with E_r(k)>0: global tokens off_k .. off_k+E_r(k)-1
  Eq. 4 tokens = (C/N)(N-1)
  Eq. 5 tokens = (N-1) * max_j sum{s : shard on j that is not the last shard of its doc}
                                                      
Bytes = tokens * Hkv * D * elem_size * 2 (K and V) per pass, * 2 for forward + backward (the
paper's factor 4).
"""

from typing import List, NamedTuple

import numpy as np

from .planner import Plan


def doc_offsets(d) -> List[int]:
    off = [0]
    for x in d:
        off.append(off[-1] + int(x))
    return off


def prefix_end(p: Plan, rank: int) -> List[int]:
    """E_r(k) for every document k."""
    E = [0] * len(p.d)
    for s in p.shards:
        if s.rank == rank:
            E[s.doc] = max(E[s.doc], s.start + s.len)
    return E


def gather_index(p: Plan, rank: int) -> np.ndarray:
    """Global token index of every row of the rank's gathered KV buffer, int32."""
    off = doc_offsets(p.d)
    E = prefix_end(p, rank)
    out = []
    for k in range(len(p.d)):
        out.extend(range(off[k], off[k] + E[k]))
    return np.asarray(out, dtype=np.int32)


def owner_of_tokens(p: Plan) -> np.ndarray:
    """Rank that holds each global token (Eq. 1: exactly one)."""
    off = doc_offsets(p.d)
    owner = np.full(off[-1], -1, dtype=np.int32)
    for s in p.shards:
        owner[off[s.doc] + s.start: off[s.doc] + s.start + s.len] = s.rank
    return owner


def q_token_index(p: Plan, rank: int) -> np.ndarray:
    """Global token index of every local query row: the rank's shards in (doc, start) order."""
    off = doc_offsets(p.d)
    out = []
    for s in p.shards:                      # canonical order is (rank, doc, start)
        if s.rank == rank:
            out.extend(range(off[s.doc] + s.start, off[s.doc] + s.start + s.len))
    return np.asarray(out, dtype=np.int32)


class KVStats(NamedTuple):
    eq4_tokens: int
    eq5_tokens: int
    gathered: tuple     # per rank: rows of the gathered buffer (local + remote)
    remote: tuple       # per rank: gathered rows owned by another rank
    nonlast: tuple      # per rank: sum of s over shards in S-hat


def kv_stats(p: Plan) -> KVStats:
    N = p.n_ranks
    C = sum(p.d)
    owner = owner_of_tokens(p)
    gathered, remote, nonlast = [], [], []
    for r in range(N):
        idx = gather_index(p, r)
        gathered.append(int(idx.size))
        remote.append(int(np.count_nonzero(owner[idx] != r)))
        nonlast.append(sum(s.len for s in p.shards
                           if s.rank == r and s.start + s.len != p.d[s.doc]))
    return KVStats((C // N) * (N - 1), (N - 1) * max(nonlast),
                   tuple(gathered), tuple(remote), tuple(nonlast))


class RankLayout(NamedTuple):
    """Varlen descriptors of one rank (SURVEY.md section 8(b) fcp_rank_layout)."""
    cu_seqlens_q: np.ndarray   # [ns+1] local query row offsets of the rank's shards
    q_pos_off: np.ndarray      # [ns]   p_i of each shard
    shard_seg: np.ndarray      # [ns]   KV segment (index among the rank's documents) of each shard
    cu_seqlens_k: np.ndarray   # [nseg+1] row offsets of the KV segments in the gathered buffer
    kv_src_start: np.ndarray   # [nseg] global token offset off_k of each segment
    kv_len: np.ndarray         # [nseg] E_r(k)
    seg_doc: np.ndarray        # [nseg] document id of each segment


def rank_layout(p: Plan, rank: int) -> RankLayout:
    off = doc_offsets(p.d)
    E = prefix_end(p, rank)
    seg_of_doc = {}
    kv_src, kv_len, seg_doc = [], [], []
    for k in range(len(p.d)):
        if E[k] > 0:
            seg_of_doc[k] = len(kv_src)
            kv_src.append(off[k])
            kv_len.append(E[k])
            seg_doc.append(k)
    cu_q, ppos, sseg = [0], [], []
    for s in p.shards:
        if s.rank == rank:
            cu_q.append(cu_q[-1] + s.len)
            ppos.append(s.start)
            sseg.append(seg_of_doc[s.doc])
    cu_k = [0]
    for x in kv_len:
        cu_k.append(cu_k[-1] + x)
    i32 = lambda a: np.asarray(a, dtype=np.int32)
    return RankLayout(i32(cu_q), i32(ppos), i32(sseg), i32(cu_k), i32(kv_src), i32(kv_len),
                      i32(seg_doc))


def scatter_add(p: Plan, rank: int, dkv_rank: np.ndarray, dKV_global: np.ndarray) -> None:
    """dKV reduction of one rank (the gradients of the communicated KV are
    reduce-scattered back to the ranks that own the tokens; the inverse of the KV selection of
    PAPER.md:111-113).  `dkv_rank` [n_kv_r, Hkv, D] holds the rank's own contribution in
    gathered-KV order; row i is added to row gather_index(p, rank)[i] of `dKV_global`
    [C, Hkv, D], in place.  Plain definition: global dK = sum over ranks of this scatter-add."""
    gi = gather_index(p, rank)
    if dkv_rank.shape[0] != gi.shape[0]:
        raise ValueError("dkv_rank has %d rows, the rank gathers %d" % (dkv_rank.shape[0], gi.shape[0]))
    # the gathered rows of one rank are distinct tokens, so a plain indexed add is exact
    dKV_global[gi] += dkv_rank


# ---------------------------------------------------------------------------------------------
# Local / prefix split of a rank's keys.
#
# PAPER.md:15 and PAPER.md:234 describe the communication-hiding alternative FlashCP is compared
# with: compute on the keys a worker already holds while the others travel, then aggregate the
# partial results.  The split used here is per shard (k, p, s) of the rank:
#   LOCAL  piece: the shard's own tokens  [p, p+s)   — causal inside the shard;
#   PREFIX piece: the tokens before it    [0, p)     — every key visible to every row.
# The two key sets are disjoint and their union is the prefix [0, p+s) the row-wise definition
# needs, so merging the two partial attentions (attention.merge) gives exactly
# the unsplit result.  Each shard is its own KV segment in both pieces; a prefix that another
# shard of the same rank also needs appears once per shard in the PREFIX buffer.
# ---------------------------------------------------------------------------------------------
PIECE_LOCAL = 1
PIECE_PREFIX = 2


def piece_layout(p: Plan, rank: int, piece: int) -> RankLayout:
    """Varlen descriptors of one piece: one KV segment per shard of the rank (seg_doc = the
    shard's document); q_pos_off is relative to the segment's first key."""
    if piece not in (PIECE_LOCAL, PIECE_PREFIX):
        raise ValueError("piece")
    off = doc_offsets(p.d)
    cu_q, ppos, sseg, cu_k, kv_src, kv_len, seg_doc = [0], [], [], [0], [], [], []
    for s in p.shards:
        if s.rank != rank:
            continue
        cu_q.append(cu_q[-1] + s.len)
        sseg.append(len(kv_src))
        if piece == PIECE_LOCAL:
            ppos.append(0)                         # row t sees keys 0..t of its own shard
            kv_src.append(off[s.doc] + s.start)
            kv_len.append(s.len)
        else:
            ppos.append(s.start)                   # row t sees keys j <= p + t, all j < p
            kv_src.append(off[s.doc])
            kv_len.append(s.start)
        seg_doc.append(s.doc)
        cu_k.append(cu_k[-1] + kv_len[-1])
    i32 = lambda a: np.asarray(a, dtype=np.int32)
    return RankLayout(i32(cu_q), i32(ppos), i32(sseg), i32(cu_k), i32(kv_src), i32(kv_len),
                      i32(seg_doc))


def piece_gather_index(p: Plan, rank: int, piece: int) -> np.ndarray:
    """Global token index of every row of the piece's KV buffer, int32."""
    L = piece_layout(p, rank, piece)
    out = []
    for a, n in zip(L.kv_src_start, L.kv_len):
        out.extend(range(int(a), int(a) + int(n)))
    return np.asarray(out, dtype=np.int32)


def piece_remote_tokens(p: Plan, rank: int, piece: int) -> int:
    """Distinct tokens of the piece's buffer that another rank owns: what a CP group would have
    to deliver before the piece can run (0 for LOCAL; for PREFIX the same tokens as the unsplit
    gather's remote part, each counted once however many shards repeat it)."""
    idx = np.unique(piece_gather_index(p, rank, piece))
    return int((owner_of_tokens(p)[idx] != rank).sum()) if idx.size else 0
