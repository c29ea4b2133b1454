"""Helpers for the GPU parity tests: run one virtual rank through the C-ABI (via the binding)
and through the oracle on the same seeded inputs, and compare element by element."""
import math

import numpy as np

import fcp_inputs
from oracle import attention as OA
from oracle import kvselect as OKV
from oracle import planner as OP

# tolerances from BASELINE.json:north_star (bf16 inputs, fp32 accumulate)
TOL_MAX_ABS = 2e-2
TOL_MEAN_ABS = 2e-3
TOL_LSE = 1e-3


def to_f64(t):
    return fcp_inputs.bf16_to_f64(t) if str(t.dtype) == "torch.bfloat16" else \
        t.detach().cpu().double().numpy()


def bf16_half_ulp(x):
    """Largest error of rounding x to bf16 (8 significant bits): 2^(floor(log2|x|) - 8)."""
    ax = np.abs(np.asarray(x, dtype=np.float64))
    e = np.floor(np.log2(np.maximum(ax, 2.0 ** -126)))
    return np.where(ax > 0, 2.0 ** (e - 8), 0.0)


def check(name, got, want, max_abs=TOL_MAX_ABS, mean_abs=TOL_MEAN_ABS, bf16_sum=False):
    """north_star tolerances.  bf16_sum=True is for dk/dv written as bf16: they are sums over
    many queries and G heads whose magnitude exceeds 8, where rounding the exact value to bf16
    alone costs up to 2^-5 = 3.1e-2 > 2e-2; the per-element bound is then max_abs + the bf16
    half-ulp of the expected value ("Reading: dk / dv written as bf16").
    The fp32-output mode of the same kernel is held to the plain max_abs."""
    got, want = np.asarray(got, dtype=np.float64), np.asarray(want, dtype=np.float64)
    assert got.shape == want.shape, (name, got.shape, want.shape)
    assert np.isfinite(got).all(), "%s: non-finite values" % name
    err = np.abs(got - want)
    mx, mean = (float(err.max()), float(err.mean())) if err.size else (0.0, 0.0)
    bound = max_abs + (bf16_half_ulp(want) if bf16_sum else 0.0)
    worst = float((err - bound).max()) if err.size else -1.0
    assert worst <= 0 and mean <= mean_abs, \
        "%s: max-abs %.3e (tol %.1e%s), mean-abs %.3e (tol %.1e)" % (
            name, mx, max_abs, " + bf16 half-ulp" if bf16_sum else "", mean, mean_abs)
    return mx, mean


def check_lse(name, got, want):
    got, want = np.asarray(got, dtype=np.float64), np.asarray(want, dtype=np.float64)
    inf = np.isneginf(want)
    assert np.array_equal(np.isneginf(got), inf), "%s: -inf pattern differs" % name
    err = np.abs(got[~inf] - want[~inf])
    mx = float(err.max()) if err.size else 0.0
    assert mx <= TOL_LSE, "%s: max-abs %.3e (tol %.1e)" % (name, mx, TOL_LSE)
    return mx


def run_rank_gpu(fcp, plan, rank, Q, K, V, dO, scale, do_bwd=True, dkv_f32=False):
    """Whole per-rank hot path on the GPU: gather -> fwd -> bwd.  Q,K,V,dO global bf16 cuda."""
    import torch
    lay = plan.rank_layout(rank)
    qi = torch.from_numpy(lay["q_token_index"].astype(np.int64)).to(Q.device)
    q, do = Q[qi].contiguous(), dO[qi].contiguous()
    kg, vg, counts = plan.kv_gather(rank, K, V)
    sched = plan.sched(rank, Q.shape[1], K.shape[1], Q.shape[2]).upload(Q.device)
    o, lse = sched.attn_fwd(q, kg, vg, scale)
    out = {"q": q, "do": do, "k": kg, "v": vg, "o": o, "lse": lse, "counts": counts,
           "layout": lay, "sched": sched}
    if do_bwd:
        out["dq"], out["dk"], out["dv"] = sched.attn_bwd(
            q, kg, vg, o, lse, do, scale, dkv_dtype=torch.float32 if dkv_f32 else torch.bfloat16)
    torch.cuda.synchronize()
    return out


def run_rank_split_gpu(fcp, plan, rank, Q, K, V, dO, scale, dK, dV):
    """The same path with the rank's keys split into the LOCAL and the PREFIX piece (include/fcp.h
    section 2b): two forwards + fcp_merge, two backwards that share one fp32 dq accumulator,
    dk / dv of both pieces scatter-added into the global fp32 dK, dV."""
    import torch
    Hq, Hkv, D = Q.shape[1], K.shape[1], Q.shape[2]
    lay = plan.rank_layout(rank)
    qi = torch.from_numpy(lay["q_token_index"].astype(np.int64)).to(Q.device)
    q, do = Q[qi].contiguous(), dO[qi].contiguous()
    part = {}
    for piece in (fcp.PIECE_LOCAL, fcp.PIECE_PREFIX):
        k, v, counts = plan.kv_gather(rank, K, V, piece=piece)
        sched = plan.sched(rank, Hq, Hkv, D, piece).upload(Q.device)
        o, lse = sched.attn_fwd(q, k, v, scale)
        part[piece] = dict(k=k, v=v, counts=counts, sched=sched, o=o, lse=lse)
    loc, pre = part[fcp.PIECE_LOCAL], part[fcp.PIECE_PREFIX]
    o, lse = fcp.merge(loc["o"], loc["lse"], pre["o"], pre["lse"])
    acc = loc["sched"].dq_accumulator(Q.device)
    acc.fill_(float("nan"))                       # the first piece must zero it itself
    dq0, loc["dk"], loc["dv"] = loc["sched"].attn_bwd(
        q, loc["k"], loc["v"], o, lse, do, scale, dkv_dtype=torch.float32, dq_accum=acc,
        dq_flags=fcp.DQ_NO_OUTPUT)
    assert dq0 is None
    dq, pre["dk"], pre["dv"] = pre["sched"].attn_bwd(
        q, pre["k"], pre["v"], o, lse, do, scale, dkv_dtype=torch.float32, dq_accum=acc,
        dq_flags=fcp.DQ_KEEP)
    for piece in (fcp.PIECE_LOCAL, fcp.PIECE_PREFIX):
        part[piece]["scatter"] = plan.kv_scatter_add(rank, part[piece]["dk"], part[piece]["dv"],
                                                     dK, dV, piece=piece)
    torch.cuda.synchronize()
    return {"o": o, "lse": lse, "dq": dq, "layout": lay, "local": loc, "prefix": pre}


def run_rank_oracle(d, N, rank, Q, K, V, dO, scale, r_ppm=1_050_000, strategy=0, do_bwd=True):
    """Same rank through oracle/ (fp64).  Q,K,V,dO are numpy fp64 arrays in global order."""
    pl = OP.plan(d, N, r_ppm, strategy)
    lay = OKV.rank_layout(pl, rank)
    qi = OKV.q_token_index(pl, rank)
    gi = OKV.gather_index(pl, rank)
    args = (lay.cu_seqlens_q, lay.q_pos_off, lay.shard_seg, lay.cu_seqlens_k, scale)
    o, lse = OA.rank_fwd(Q[qi], K[gi], V[gi], *args)
    out = {"o": o, "lse": lse, "gather_index": gi, "q_index": qi}
    if do_bwd:
        out["dq"], out["dk"], out["dv"] = OA.rank_bwd(Q[qi], K[gi], V[gi], o, lse, dO[qi], *args)
    return out


def compare_rank(fcp, d, N, rank, Hq, Hkv, D, seed=0, r_ppm=1_050_000, strategy=0, do_bwd=True,
                 verbose=False, dkv_f32=False):
    import torch
    C = sum(d)
    scale = 1.0 / math.sqrt(D)
    Q, K, V, dO = fcp_inputs.make_tensors(C, Hq, Hkv, D, seed)
    plan = fcp.Plan(d, N, r_ppm, strategy)
    dev = torch.device("cuda:0")
    g = run_rank_gpu(fcp, plan, rank, Q.to(dev), K.to(dev), V.to(dev), dO.to(dev), scale, do_bwd,
                     dkv_f32)
    w = run_rank_oracle(d, N, rank, to_f64(Q), to_f64(K), to_f64(V), to_f64(dO), scale, r_ppm,
                        strategy, do_bwd)
    # gathered KV: bit-exact
    assert torch.equal(g["k"].cpu(), K[torch.from_numpy(w["gather_index"].astype(np.int64))])
    assert torch.equal(g["v"].cpu(), V[torch.from_numpy(w["gather_index"].astype(np.int64))])
    res = {"o": check("o", to_f64(g["o"]), w["o"]), "lse": check_lse("lse", to_f64(g["lse"]), w["lse"])}
    if do_bwd:
        res["dq"] = check("dq", to_f64(g["dq"]), w["dq"])
        for k in ("dk", "dv"):
            res[k] = check(k, to_f64(g[k]), w[k], bf16_sum=not dkv_f32)
    if verbose:
        print("rank", rank, res)
    return res
