"""N > 1 path of bench.py on CPU: two gloo ranks (no GPU).  The hot path shards over GPUs as
independent packed batches (weak scaling, no data-path collective — DESIGN.md section 6); what
crosses ranks is only the timing / flop aggregation, which is what these tests exercise, plus
the host planner running in both processes on their own batch."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    import fcp_inputs
    import paper_2606_08476_b200 as fcp
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # every rank plans its own packed batch (seed + rank), as run_fcp does
        cfg = fcp_inputs.CONFIGS["8b"]
        d = fcp_inputs.doc_lengths("8b", bench.rank_seed(0, rank))
        plan = fcp.Plan(d, cfg.N)
        st = plan.stats()
        assert st["context_len"] == cfg.C and st["tokens_per_rank"] == cfg.C // cfg.N
        f_fwd, f_bwd = bench.useful_flops(cfg, d)
        my_flops = float(f_fwd + f_bwd)
        my_ms = 10.0 * (rank + 1)                    # rank 1 is the slow one
        value, ms = bench.job_throughput(my_flops, my_ms, dist, "cpu")
        total = bench.over_ranks(my_flops, "sum", dist, "cpu")
        n_docs_max = bench.over_ranks(float(len(d)), "max", dist, "cpu")
        out.put((rank, value, ms, total, my_flops, len(d), n_docs_max))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_aggregate_whole_job_throughput():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, v0, ms0, tot0, f0, n0, nm0), (_, v1, ms1, tot1, f1, n1, nm1) = res
    # time = max over ranks, work = sum over ranks, identical on both ranks
    assert ms0 == ms1 == 20.0
    assert tot0 == tot1 == pytest.approx(f0 + f1)
    assert v0 == v1 == pytest.approx((f0 + f1) / 20e-3 / 1e12)
    # the two ranks really worked on different batches
    assert (f0, n0) != (f1, n1)
    assert nm0 == nm1 == max(n0, n1)


def test_single_process_is_identity():
    import bench
    assert bench.over_ranks(3.5, "max") == 3.5
    v, ms = bench.job_throughput(2e12, 1000.0)
    assert ms == 1000.0 and v == pytest.approx(2.0)


# ------------------------------------------------------------------------------------------
# KV exchange of a real CP group (paper_2606_08476_b200/exchange.py) on gloo ranks
# ------------------------------------------------------------------------------------------
_XCASES = {
    2: ([700, 90, 300, 190], 0),          # Per-Doc pair + whole documents
    4: ([2048, 37, 1, 600, 130, 256], 0),  # long document split over all ranks, 1-token document
}


def _xchg_grads(n_rows, Hkv, D, r):
    import torch
    g = torch.Generator().manual_seed(1000 + r)
    return (torch.randn((n_rows, Hkv, D), generator=g), torch.randn((n_rows, Hkv, D), generator=g))


def _xchg_worker(rank, world, port, out):
    import numpy as np
    import torch
    import torch.distributed as dist
    import fcp_inputs
    import paper_2606_08476_b200 as fcp
    from paper_2606_08476_b200.exchange import KVExchange
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        d, strategy = _XCASES[world]
        Hkv, D = 2, 64
        _, K, V, _ = fcp_inputs.make_tensors(sum(d), 2, Hkv, D, 3)
        plan = fcp.Plan(d, world, strategy=strategy)
        x = KVExchange(plan, rank)
        lay = plan.rank_layout(rank)
        qi = torch.from_numpy(lay["q_token_index"].astype(np.int64))
        k, v = x.gather(K[qi].contiguous(), V[qi].contiguous())      # this rank holds only its rows
        dk_r, dv_r = _xchg_grads(x.n_kv, Hkv, D, rank)
        dk_l, dv_l = x.scatter_add(dk_r, dv_r)
        out.put((rank, k.view(torch.int16).numpy(), v.view(torch.int16).numpy(), dk_l.numpy(),
                 dv_l.numpy(), x.remote_tokens, plan.rank_stats(rank)["remote_tokens"]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 4])
def test_kv_exchange_matches_oracle_gather_and_scatter(world):
    """Each gloo rank starts with its own K, V rows only; after the all-to-all-v it holds exactly
    the rows the ORACLE's gather index names (bit-exact), having received exactly the planner's
    remote-token count; the way back sums every rank's dk, dv rows onto their owners as the
    oracle's token-by-token scatter does."""
    import numpy as np
    import torch
    import torch.multiprocessing as mp
    import fcp_inputs
    from oracle import kvselect as KV
    from oracle import planner as P
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_xchg_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((out.get(timeout=240) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    d, strategy = _XCASES[world]
    Hkv, D = 2, 64
    _, K, V, _ = fcp_inputs.make_tensors(sum(d), 2, Hkv, D, 3)
    Ki, Vi = K.view(torch.int16).numpy(), V.view(torch.int16).numpy()
    pl = P.plan(d, world, 1_050_000, strategy)
    kst = KV.kv_stats(pl)
    dK = np.zeros((sum(d), Hkv, D))
    dV = np.zeros_like(dK)
    for r in range(world):                                  # rank order, one add per element and rank
        gi = KV.gather_index(pl, r)
        gk, gv = _xchg_grads(len(gi), Hkv, D, r)
        dK[gi] += gk.double().numpy()
        dV[gi] += gv.double().numpy()
    for r, k, v, dk_l, dv_l, remote, remote_plan in res:
        gi = KV.gather_index(pl, r)
        assert np.array_equal(k, Ki[gi]) and np.array_equal(v, Vi[gi])
        assert remote == remote_plan == kst.remote[r]
        qi = KV.q_token_index(pl, r)
        assert np.abs(dk_l - dK[qi]).max() < 1e-5 and np.abs(dv_l - dV[qi]).max() < 1e-5
    assert sum(t[5] for t in res) > 0                       # the case really moves rows


def test_bench_spawns_its_ranks_when_no_launcher_is_present():
    """`python bench.py --gpus N` without WORLD_SIZE re-executes itself under
    torch.distributed.run with N processes (the flag used to be ignored).  Exercised on
    the CPU through the reference arm: rank 0 alone prints the JSON line, the other rank exits 0;
    a launcher whose WORLD_SIZE contradicts --gpus is refused by the fcp arm."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--config", "tiny"], cwd=root, env=env,
                       stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, timeout=300)
    assert r.returncode == 0, r.stdout[-2000:]
    lines = [json.loads(x) for x in r.stdout.splitlines() if x.startswith("{")]
    assert len(lines) == 1 and lines[0]["impl"] == "reference" and lines[0]["n_gpus"] == 2
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "1"],
                       cwd=root, env=dict(env, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0"),
                       stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, timeout=300)
    assert r.returncode != 0 and ("--gpus 2 but WORLD_SIZE=1" in r.stdout or "CUDA device" in r.stdout)
