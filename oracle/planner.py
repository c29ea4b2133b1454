"""Oracle: FlashCP sharding planner (TEST INFRASTRUCTURE, see oracle/__init__.py).

Follows PAPER.md section 3.1 (problem statement, Eq. 1-3, W_i at PAPER.md:101), section 3.3
(Whole-Doc / Per-Doc) and Algorithm 1 step by step in the
deterministic reading listed in DESIGN.md section 3 ("readings of the paper").  Integer arithmetic only.

Notation: documents D=[d_1..d_n] (0-based ``d[k]`` here), CP size N, context
C = sum d, a shard = (doc, start p, len s, rank j); W = (2p+s+1)*s/2.
"""

from typing import List, NamedTuple, Sequence

STRATEGY_HYBRID = 0      # Algorithm 1
STRATEGY_ALL_PER_DOC = 1  # every document Per-Doc
STRATEGY_WHOLE_DOC = 2   # Whole-Doc only, never Per-Doc
STRATEGY_PER_SEQ = 3     # Llama3 CP baseline: the packed SEQUENCE in 2N chunks

DEFAULT_R_PPM = 1_050_000  # R = 1.05 (paper gives no value; its heuristic reaches 1.04)


class Shard(NamedTuple):
    doc: int
    start: int   # p_i, tokens of the document preceding the shard
    len: int     # s_i
    rank: int    # j with x_ij = 1 (Eq. 1)


class Plan(NamedTuple):
    d: tuple            # document lengths, original packed order
    n_ranks: int
    shards: tuple       # canonical: sorted by (rank, doc, start), contiguous neighbours merged
    per_doc: tuple      # document ids sharded Per-Doc, in the order Algorithm 1 popped them
    pass_ratios: tuple  # (max_load, sum_load) after each pass of the while loop


def W(p: int, s: int) -> int:
    """Attention workload of a shard with prefix p and length s."""
    return (2 * p + s + 1) * s // 2


def _argmin(keys):
    best = None
    for j, key in enumerate(keys):
        if key is not None and (best is None or key < keys[best]):
            best = j
    return best


def plan(d: Sequence[int], n_ranks: int, r_ppm: int = DEFAULT_R_PPM,
         strategy: int = STRATEGY_HYBRID, align: int = 1) -> Plan:
    """Algorithm 1.  Raises ValueError where the C-ABI returns INVALID_ARG.

    align = A > 1 selects the tile-aligned variant (the paper only notes
    that short / ragged shards cost kernel efficiency): cuts are placed on
    multiples of A document positions wherever Eq. 2 leaves the choice, so that a shard's query
    tiles line up with the key tiles of its document.  A = 1 is Algorithm 1 as read above, step
    for step.  With A > 1 (readings of DESIGN.md section 2.3):
      Per-Doc   chunk length q = (d div 2NA) A; of the leftover L = d - 2Nq the aligned part
                h = (L div A) A is the head item [0, h) of the Whole-Doc pool, chunks start at
                h + c q, and the last e = L - h < A tokens are a movable item [d - e, d) that
                starts on the worker of the LAST chunk (worker 0: it merges with that chunk,
                which ends at the document's ragged end anyway, unless the equal-token repair
                has to move it); q = 0 leaves the document whole.
      repair    handing g tokens from worker a to b when no whole item fits:
                g >= A: cut (g div A) A tokens from the head of a's longest item that starts on
                a multiple of A (none: its longest item, g tokens);
                g <  A: cut g tokens from the head of a's SHORTEST item (the unaligned cut that
                Eq. 2 forces lands on a short document, where a ragged tile wastes least)."""
    d = [int(x) for x in d]
    n, N, A = len(d), int(n_ranks), int(align)
    if n < 1 or N < 1 or any(x < 1 for x in d) or r_ppm < 1_000_000 or A < 1:
        raise ValueError("invalid argument")
    if strategy not in (STRATEGY_HYBRID, STRATEGY_ALL_PER_DOC, STRATEGY_WHOLE_DOC,
                        STRATEGY_PER_SEQ):
        raise ValueError("invalid strategy")
    C = sum(d)
    if C % N != 0:                       # Eq. 2 needs C/N integral
        raise ValueError("C not divisible by N")
    T = C // N

    if strategy == STRATEGY_PER_SEQ:
        return _per_seq(d, N, C)

    # line 1: sort D in descending order of length (ties: lower id first)
    order = sorted(range(n), key=lambda k: (-d[k], k))

    if strategy == STRATEGY_ALL_PER_DOC:
        k_first, k_last = n, n
    elif strategy == STRATEGY_WHOLE_DOC:
        k_first, k_last = 0, 0
    else:
        k_first, k_last = 0, n

    pass_ratios = []
    k_per = k_first
    while True:                                        # line 4: while Cur_R > R
        tok = [0] * N
        load = [0] * N
        fixed = []                                     # Per-Doc chunk shards (never moved)
        items = [[] for _ in range(N)]                 # movable Whole-Doc items [doc, start, len]
        pool = []
        # Per_Doc_P: 2N chunks, chunks c and 2N-1-c to worker c
        for i in order[:k_per]:
            q = d[i] // (2 * N * A) * A                 # A = 1: d div 2N
            if q == 0:
                pool.append([i, 0, d[i]])
                continue
            r = (d[i] - 2 * N * q) // A * A             # head of the document; A = 1: d mod 2N
            e = d[i] - 2 * N * q - r                    # < A tokens on the last chunk; A = 1: 0
            if r > 0:
                pool.append([i, 0, r])
            for c in range(2 * N):
                j = c if c < N else 2 * N - 1 - c
                fixed.append(Shard(i, r + c * q, q, j))
                tok[j] += q
                load[j] += W(r + c * q, q)
            if e > 0:                                   # only with A > 1
                items[0].append([i, d[i] - e, e])
                tok[0] += e
                load[0] += W(d[i] - e, e)
        for i in order[k_per:]:
            pool.append([i, 0, d[i]])
        pool.sort(key=lambda it: (-it[2], it[0]))
        # lines 5-9: add each document to the least-loaded worker (by workload)
        for it in pool:
            j = _argmin([(load[x], x) for x in range(N)])
            items[j].append(it)
            tok[j] += it[2]
            load[j] += W(it[1], it[2])
        # lines 10-16: make Eq. 2 hold by Whole-Doc sharding
        while True:
            a = _argmin([(-tok[x], x) for x in range(N)])   # most tokens, ties lowest rank
            if tok[a] == T:
                break
            e = tok[a] - T
            while e > 0:
                b = _argmin([(load[x], x) if tok[x] < T else None for x in range(N)])
                g = min(e, T - tok[b])
                fit = [it for it in items[a] if it[2] <= g]
                if fit:                                  # move a whole item: zero communication
                    x = min(fit, key=lambda it: (it[2], it[0]))
                    items[a].remove(x)
                    moved = x
                else:                                    # cut the head ("lower segment",
                    # PAPER.md:124) of the longest item; its tail stays on worker a
                    if g >= A:
                        on_grid = [it for it in items[a] if it[1] % A == 0]
                        x = min(on_grid or items[a], key=lambda it: (-it[2], it[0]))
                        if on_grid:
                            g = g // A * A
                    else:                                # only with A > 1: the ragged remainder
                        x = min(items[a], key=lambda it: (it[2], it[0]))
                    moved = [x[0], x[1], g]
                    x[1] += g
                    x[2] -= g
                m = moved[2]
                w_moved = W(moved[1], m)                 # W(p,s) adds over a cut: W(p,a+b)=W(p,a)+W(p+a,b)
                load[a] -= w_moved
                tok[a] -= m
                items[b].append(moved)
                load[b] += w_moved
                tok[b] += m
                e -= m
        # line 18: Cur_R = max/avg workload over all CP workers
        max_load, sum_load = max(load), sum(load)
        pass_ratios.append((max_load, sum_load))
        over = max_load * N * 1_000_000 > r_ppm * sum_load
        if not over or k_per >= k_last:
            break
        k_per += 1                                      # lines 19-23: longest doc -> Per-Doc

    shards = list(fixed)
    for j in range(N):
        for it in items[j]:
            shards.append(Shard(it[0], it[1], it[2], j))
    shards.sort(key=lambda s: (s.rank, s.doc, s.start))
    merged: List[Shard] = []
    for s in shards:                                    # merge contiguous neighbours on one rank
        if merged and merged[-1].rank == s.rank and merged[-1].doc == s.doc \
                and merged[-1].start + merged[-1].len == s.start:
            last = merged.pop()
            merged.append(Shard(s.doc, last.start, last.len + s.len, s.rank))
        else:
            merged.append(s)
    return Plan(tuple(d), N, tuple(merged), tuple(order[:k_per]), tuple(pass_ratios))


def _per_seq(d: List[int], N: int, C: int) -> Plan:
    """Per-Sequence sharding, the Llama3 CP baseline the paper compares with (Fig.
    1(b), Fig. 2): the packed sequence of C tokens is split into 2N equal chunks regardless of
    document borders and worker i processes chunks i and 2N-1-i.  A chunk that spans several
    documents yields one shard per document piece.  Needs C % 2N == 0 (equal chunks; reading
    listed in DESIGN.md section 2.3).  No Per-Doc set, a single pass."""
    if C % (2 * N) != 0:
        raise ValueError("C not divisible by 2N")
    q = C // (2 * N)
    off = [0]
    for x in d:
        off.append(off[-1] + x)
    shards = []
    for c in range(2 * N):
        j = c if c < N else 2 * N - 1 - c
        lo, hi = c * q, (c + 1) * q
        for k, x in enumerate(d):                       # pieces of documents inside [lo, hi)
            a, b = max(lo, off[k]), min(hi, off[k + 1])
            if a < b:
                shards.append(Shard(k, a - off[k], b - a, j))
    shards.sort(key=lambda s: (s.rank, s.doc, s.start))
    merged: List[Shard] = []
    for s in shards:
        if merged and merged[-1].rank == s.rank and merged[-1].doc == s.doc \
                and merged[-1].start + merged[-1].len == s.start:
            last = merged.pop()
            merged.append(Shard(s.doc, last.start, last.len + s.len, s.rank))
        else:
            merged.append(s)
    load = [0] * N
    for s in merged:
        load[s.rank] += W(s.start, s.len)
    return Plan(tuple(d), N, tuple(merged), (), ((max(load), sum(load)),))


def rank_tokens(p: Plan) -> List[int]:
    """Left side of Eq. 2 for every worker."""
    out = [0] * p.n_ranks
    for s in p.shards:
        out[s.rank] += s.len
    return out


def rank_loads(p: Plan) -> List[int]:
    """Inner sum of Eq. 3 for every worker."""
    out = [0] * p.n_ranks
    for s in p.shards:
        out[s.rank] += W(s.start, s.len)
    return out


def imbalance_ppm(p: Plan) -> int:
    """floor(1e6 * max_workload / avg_workload)."""
    loads = rank_loads(p)
    return max(loads) * p.n_ranks * 1_000_000 // sum(loads)
