"""KV exchange of a real context-parallel group over torch.distributed (SURVEY.md 8(e) and 8(f)
NEXT 1; PAPER.md:72, 113 — "gather only the KV of preceding tokens of documents whose queries
live on the rank" — and PAPER.md:109, 204 for the dKV reduction on the way back).

On one GPU the CP ranks are virtual and `fcp_kv_gather` / `fcp_kv_scatter_add` move the rows
device-locally.  With one process per GPU every rank holds only its own shards' K, V rows (in its
local query order, `rank_layout()["q_token_index"]`), and what the plan makes it gather from other
ranks has to travel.  Instead of the paper's AllGather of every rank's non-last shards (Eq. 5)
followed by a copy, this is the all-to-all-v the plan defines exactly: rank s sends rank r the rows
of the tokens r needs and s owns — `remote_tokens` rows arrive at r, not one more (NVSwitch gives
every pair of GPUs full bandwidth, so the grouped send/recv costs what its bytes cost).  Every
rank derives all split sizes from the deterministic host plan; nothing but the rows is exchanged.

The transport is `torch.distributed.all_to_all_single` (NCCL over NVLink on GPUs, gloo in the CPU
tests); packing and unpacking are index copies on the tensors' device.  K and V travel in one
collective.  This module is plumbing around the C ABI, not part of the timed hot path."""
import numpy as np


class KVExchange:
    """Split sizes and row indices of one rank's part in the exchange of one plan."""

    def __init__(self, plan, rank):
        N = plan.n_ranks
        lays = [plan.rank_layout(r) for r in range(N)]
        C = sum(len(l["q_token_index"]) for l in lays)
        owner = np.full(C, -1, dtype=np.int64)
        local_row = np.zeros(C, dtype=np.int64)
        for s, l in enumerate(lays):
            qi = l["q_token_index"].astype(np.int64)
            owner[qi] = s
            local_row[qi] = np.arange(len(qi))
        assert (owner >= 0).all()                      # Eq. 1: every token is owned by one rank
        self.rank, self.world = rank, N
        self.n_local = len(lays[rank]["q_token_index"])
        need = lays[rank]["kv_token_index"].astype(np.int64)      # gathered order of this rank
        self.n_kv = len(need)
        src = owner[need]
        # receive side: where the rows of source rank s go in the gathered buffer (s ascending,
        # inside a source in gathered order)
        self.recv_pos = [np.nonzero(src == s)[0] for s in range(N)]
        self.recv_counts = [int(len(p)) for p in self.recv_pos]
        # send side: my local rows that rank r gathers, in r's gathered order
        self.send_rows = []
        for r in range(N):
            need_r = lays[r]["kv_token_index"].astype(np.int64)
            self.send_rows.append(local_row[need_r[owner[need_r] == rank]])
        self.send_counts = [int(len(x)) for x in self.send_rows]
        self.remote_tokens = self.n_kv - self.recv_counts[rank]

    def _idx(self, arrays, device):
        import torch
        return torch.from_numpy(np.concatenate(arrays).astype(np.int64)).to(device)

    def gather(self, k_local, v_local, group=None):
        """k_local, v_local [n_local, Hkv, D] (this rank's rows) -> k, v [n_kv, Hkv, D] in the
        layout fcp_kv_gather produces (what fcp_attn_fwd / fcp_attn_bwd read)."""
        import torch
        import torch.distributed as dist
        assert k_local.shape == v_local.shape and k_local.shape[0] == self.n_local
        kv = torch.stack((k_local, v_local), dim=1)                # [n_local, 2, Hkv, D]
        send = kv.index_select(0, self._idx(self.send_rows, kv.device)).contiguous()
        recv = torch.empty((self.n_kv,) + tuple(kv.shape[1:]), dtype=kv.dtype, device=kv.device)
        # bytes are bytes: the rows travel as uint8 (gloo has no bf16 all-to-all)
        dist.all_to_all_single(recv.view(torch.uint8), send.view(torch.uint8), self.recv_counts,
                               self.send_counts, group=group)
        out = torch.empty_like(recv)
        out.index_copy_(0, self._idx(self.recv_pos, kv.device), recv)
        return out[:, 0].contiguous(), out[:, 1].contiguous()

    def scatter_add(self, dk_r, dv_r, group=None):
        """The way back: dk_r, dv_r [n_kv, Hkv, D] (gradients of the gathered rows) -> fp32
        dk_local, dv_local [n_local, Hkv, D] = sum over all ranks of what they computed for the
        tokens this rank owns.  Contributions are added in source-rank order, one fp32 add per
        element and source (the recurrence fcp_kv_scatter_add uses), so the result is
        reproducible."""
        import torch
        import torch.distributed as dist
        assert dk_r.shape == dv_r.shape and dk_r.shape[0] == self.n_kv
        g = torch.stack((dk_r, dv_r), dim=1).float()
        send = g.index_select(0, self._idx(self.recv_pos, g.device)).contiguous()
        recv = torch.empty((sum(self.send_counts),) + tuple(g.shape[1:]), dtype=g.dtype,
                           device=g.device)
        dist.all_to_all_single(recv, send, self.send_counts, self.recv_counts, group=group)
        acc = torch.zeros((self.n_local,) + tuple(g.shape[1:]), dtype=torch.float32, device=g.device)
        o = 0
        for r in range(self.world):                    # rows of one source are distinct tokens
            n = self.send_counts[r]
            if n:
                rows = torch.from_numpy(self.send_rows[r]).to(g.device)
                acc.index_add_(0, rows, recv[o:o + n])
            o += n
        return acc[:, 0].contiguous(), acc[:, 1].contiguous()
