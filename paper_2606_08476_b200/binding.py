"""Thin ctypes binding over libfcp.so (include/fcp.h): argument marshalling only — every step
of the hot path runs in the library's kernels.  There is no CPU fallback: a missing library
or a non-zero status raises.  torch is used only for device memory and streams."""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# FCP_LIB selects another build of the same library (tests/test_sanitizers.py: the host sources
# under ASan / UBSan); there is still no fallback: the named file must exist and export every symbol
LIB_PATH = os.environ.get("FCP_LIB") or os.path.join(_HERE, "libfcp.so")

EXPORTS = [
    "fcp_strerror", "fcp_version", "fcp_plan_create", "fcp_plan_destroy", "fcp_plan_shards",
    "fcp_plan_perdoc", "fcp_plan_stats", "fcp_plan_rank_stats", "fcp_rank_layout",
    "fcp_kv_gather", "fcp_kv_scatter_add", "fcp_sched_create", "fcp_sched_from_plan", "fcp_sched_destroy",
    "fcp_sched_workspace_size", "fcp_sched_upload", "fcp_sched_get_info", "fcp_attn_fwd",
    "fcp_attn_bwd", "fcp_merge", "fcp_plan_piece_stats", "fcp_piece_layout", "fcp_kv_gather_piece",
    "fcp_kv_scatter_add_piece", "fcp_sched_from_plan_piece", "fcp_sched_get_list",
    "fcp_kv_reduce_finish", "fcp_attn_bwd_static",
]

STRATEGY_HYBRID, STRATEGY_ALL_PER_DOC, STRATEGY_WHOLE_DOC, STRATEGY_PER_SEQ = 0, 1, 2, 3
# key sets of a rank (include/fcp.h section 2b): the whole prefix, or its local / prefix split
PIECE_FULL, PIECE_LOCAL, PIECE_PREFIX = 0, 1, 2
DQ_KEEP, DQ_NO_OUTPUT = 1, 2
TOO_LARGE = -7                               # fcp_status FCP_TOO_LARGE
STATIC_WORKSPACE_BYTES = 32 << 20            # FCP_STATIC_WORKSPACE_BYTES


class FcpError(RuntimeError):
    def __init__(self, status, what):
        self.status = status
        super().__init__("%s failed: %s (%d)" % (what, _lib().fcp_strerror(status).decode(), status))


class _Shard(C.Structure):
    _fields_ = [("doc", C.c_int32), ("start", C.c_int32), ("len", C.c_int32), ("rank", C.c_int32)]


class _PlanOpts(C.Structure):
    _fields_ = [("imbalance_ppm", C.c_int64), ("strategy", C.c_int32),
                ("align_tokens", C.c_int32)]


class _Stats(C.Structure):
    _fields_ = [("n_ranks", C.c_int32), ("n_docs", C.c_int32), ("n_shards", C.c_int32),
                ("n_per_doc", C.c_int32), ("n_passes", C.c_int32), ("reserved", C.c_int32),
                ("context_len", C.c_int64), ("tokens_per_rank", C.c_int64),
                ("max_load", C.c_uint64), ("sum_load", C.c_uint64), ("imbalance_ppm", C.c_int64),
                ("eq4_tokens", C.c_int64), ("eq5_tokens", C.c_int64),
                ("max_remote_tokens", C.c_int64), ("sum_remote_tokens", C.c_int64),
                ("max_gathered_tokens", C.c_int64), ("sum_gathered_tokens", C.c_int64)]


class _RankStats(C.Structure):
    _fields_ = [("n_shards", C.c_int32), ("n_segs", C.c_int32), ("n_q", C.c_int64),
                ("n_kv", C.c_int64), ("remote_tokens", C.c_int64), ("nonlast_tokens", C.c_int64),
                ("load", C.c_uint64)]


_I32P = C.POINTER(C.c_int32)


class _Layout(C.Structure):
    _fields_ = [(n, _I32P) for n in ("cu_seqlens_q", "q_pos_off", "shard_seg", "cu_seqlens_k",
                                     "kv_src_start", "kv_len", "q_token_index", "kv_token_index")]


class _GatherCounts(C.Structure):
    _fields_ = [("total_tokens", C.c_int64), ("remote_tokens", C.c_int64),
                ("total_bytes", C.c_int64), ("remote_bytes", C.c_int64),
                ("n_ranges", C.c_int32), ("reserved", C.c_int32)]


class _SchedInfo(C.Structure):
    _fields_ = [("n_fwd_items", C.c_int32), ("n_bwd_items", C.c_int32),
                ("fwd_kv_tiles", C.c_int64), ("bwd_tile_pairs", C.c_int64),
                ("useful_pairs", C.c_uint64), ("n_q", C.c_int64), ("n_kv", C.c_int64),
                ("n_q_pad", C.c_int64)]


class _AttnArgs(C.Structure):
    _fields_ = [("sched", C.c_void_p), ("workspace", C.c_void_p), ("q", C.c_void_p),
                ("k", C.c_void_p), ("v", C.c_void_p), ("o", C.c_void_p), ("lse", C.c_void_p),
                ("scale", C.c_float), ("dkv_dtype", C.c_int32), ("stream", C.c_void_p),
                ("ev_start", C.c_void_p), ("ev_stop", C.c_void_p), ("dq_accum", C.c_void_p),
                ("dq_flags", C.c_int32)]


_LIB = None


def _lib():
    global _LIB
    if _LIB is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libfcp.so is not built: run `python -m paper_2606_08476_b200.build` "
                              "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        lib.fcp_strerror.restype = C.c_char_p
        lib.fcp_strerror.argtypes = [C.c_int]
        lib.fcp_version.restype = C.c_char_p
        lib.fcp_plan_destroy.restype = None
        lib.fcp_plan_destroy.argtypes = [C.c_void_p]
        lib.fcp_sched_destroy.restype = None
        lib.fcp_sched_destroy.argtypes = [C.c_void_p]
        lib.fcp_plan_create.argtypes = [_I32P, C.c_int32, C.c_int32, C.POINTER(_PlanOpts),
                                        C.POINTER(C.c_void_p)]
        lib.fcp_plan_shards.argtypes = [C.c_void_p, C.c_int32, C.POINTER(_Shard), C.c_int32, _I32P]
        lib.fcp_plan_perdoc.argtypes = [C.c_void_p, _I32P, C.c_int32, _I32P]
        lib.fcp_plan_stats.argtypes = [C.c_void_p, C.POINTER(_Stats)]
        lib.fcp_plan_rank_stats.argtypes = [C.c_void_p, C.c_int32, C.POINTER(_RankStats)]
        lib.fcp_plan_piece_stats.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.POINTER(_RankStats)]
        lib.fcp_rank_layout.argtypes = [C.c_void_p, C.c_int32, C.POINTER(_Layout)]
        lib.fcp_piece_layout.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.POINTER(_Layout)]
        gather = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p,
                  C.POINTER(_GatherCounts)]
        lib.fcp_kv_gather.argtypes = [C.c_void_p, C.c_int32] + gather
        lib.fcp_kv_gather_piece.argtypes = [C.c_void_p, C.c_int32, C.c_int32] + gather
        scatter = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32,
                   C.c_void_p, C.POINTER(_GatherCounts)]
        lib.fcp_kv_scatter_add.argtypes = [C.c_void_p, C.c_int32] + scatter
        lib.fcp_kv_scatter_add_piece.argtypes = [C.c_void_p, C.c_int32, C.c_int32] + scatter
        lib.fcp_kv_reduce_finish.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                             C.c_int64, C.c_void_p]
        lib.fcp_sched_create.argtypes = [_I32P, _I32P, _I32P, C.c_int32, _I32P, C.c_int32,
                                         C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_void_p)]
        lib.fcp_sched_from_plan.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_int32,
                                            C.POINTER(C.c_void_p)]
        lib.fcp_sched_from_plan_piece.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32,
                                                  C.c_int32, C.c_int32, C.POINTER(C.c_void_p)]
        lib.fcp_sched_workspace_size.argtypes = [C.c_void_p, C.POINTER(C.c_size_t)]
        lib.fcp_sched_upload.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        lib.fcp_sched_get_info.argtypes = [C.c_void_p, C.POINTER(_SchedInfo)]
        lib.fcp_sched_get_list.argtypes = [C.c_void_p, C.c_int32, _I32P, C.c_int64,
                                           C.POINTER(C.c_int64)]
        lib.fcp_attn_fwd.argtypes = [C.POINTER(_AttnArgs)]
        lib.fcp_attn_bwd.argtypes = [C.POINTER(_AttnArgs), C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_void_p]
        lib.fcp_attn_bwd_static.argtypes = lib.fcp_attn_bwd.argtypes
        lib.fcp_merge.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                  C.c_void_p, C.c_int64, C.c_int32, C.c_int32, C.c_int32,
                                  C.c_void_p]
        _LIB = lib
    return _LIB


def _check(status, what):
    if status != 0:
        raise FcpError(status, what)


def _i32(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.int32))


def _p(a):
    return a.ctypes.data_as(_I32P)


def _struct_dict(s):
    return {n: getattr(s, n) for n, _ in s._fields_ if n != "reserved"}


def version():
    return _lib().fcp_version().decode()


def _stream_ptr(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


def _event_ptr(ev):
    """cudaEvent_t of a torch.cuda.Event (created lazily by torch: record it once first)."""
    h = getattr(ev, "cuda_event", ev)
    if not h:
        raise ValueError("torch.cuda.Event has no handle yet: call ev.record() once before use")
    return h


class Plan:
    """fcp_plan: Algorithm 1 sharding plan (host)."""

    def __init__(self, doc_lengths, n_ranks, imbalance_ppm=0, strategy=STRATEGY_HYBRID, align=0):
        d = _i32(doc_lengths)
        opts = _PlanOpts(int(imbalance_ppm), int(strategy), int(align))
        h = C.c_void_p()
        _check(_lib().fcp_plan_create(_p(d), d.size, int(n_ranks), C.byref(opts), C.byref(h)),
               "fcp_plan_create")
        self._h = h
        self.n_ranks = int(n_ranks)
        self.doc_lengths = d.copy()

    def __del__(self):
        if getattr(self, "_h", None) and _LIB is not None:   # module globals vanish at shutdown
            _LIB.fcp_plan_destroy(self._h)
            self._h = None

    def shards(self, rank=-1):
        """[(doc, start, len, rank)] canonical order."""
        n = C.c_int32()
        st = _lib().fcp_plan_shards(self._h, rank, None, 0, C.byref(n))
        if st not in (0, -3):
            _check(st, "fcp_plan_shards")
        buf = (_Shard * max(1, n.value))()
        _check(_lib().fcp_plan_shards(self._h, rank, buf, n.value, C.byref(n)), "fcp_plan_shards")
        return [(buf[i].doc, buf[i].start, buf[i].len, buf[i].rank) for i in range(n.value)]

    def per_doc(self):
        n = C.c_int32()
        st = _lib().fcp_plan_perdoc(self._h, None, 0, C.byref(n))
        if st not in (0, -3):
            _check(st, "fcp_plan_perdoc")
        buf = np.zeros(max(1, n.value), dtype=np.int32)
        _check(_lib().fcp_plan_perdoc(self._h, _p(buf), n.value, C.byref(n)), "fcp_plan_perdoc")
        return [int(x) for x in buf[:n.value]]

    def stats(self):
        s = _Stats()
        _check(_lib().fcp_plan_stats(self._h, C.byref(s)), "fcp_plan_stats")
        return _struct_dict(s)

    def rank_stats(self, rank, piece=PIECE_FULL):
        s = _RankStats()
        _check(_lib().fcp_plan_piece_stats(self._h, rank, piece, C.byref(s)), "fcp_plan_piece_stats")
        return _struct_dict(s)

    def rank_layout(self, rank, piece=PIECE_FULL):
        """dict of int32 numpy arrays (see fcp_layout in include/fcp.h)."""
        rs = self.rank_stats(rank, piece)
        ns, ng = rs["n_shards"], rs["n_segs"]
        sizes = {"cu_seqlens_q": ns + 1, "q_pos_off": ns, "shard_seg": ns, "cu_seqlens_k": ng + 1,
                 "kv_src_start": ng, "kv_len": ng, "q_token_index": rs["n_q"],
                 "kv_token_index": rs["n_kv"]}
        arrs = {k: np.zeros(max(1, v), dtype=np.int32) for k, v in sizes.items()}
        lay = _Layout(**{k: _p(a) for k, a in arrs.items()})
        _check(_lib().fcp_piece_layout(self._h, rank, piece, C.byref(lay)), "fcp_piece_layout")
        return {k: arrs[k][:sizes[k]] for k in sizes}

    def kv_gather(self, rank, K, V, k_out=None, v_out=None, stream=None, piece=PIECE_FULL):
        """Device gather of the rank's KV prefixes (or of one piece of their local / prefix
        split).  K, V: torch bf16 [C,Hkv,D] on the GPU.  Returns (k_out, v_out, counts)."""
        import torch
        assert K.is_cuda and V.is_cuda and K.is_contiguous() and V.is_contiguous()
        Hkv, D = K.shape[1], K.shape[2]
        n_kv = self.rank_stats(rank, piece)["n_kv"]
        if k_out is None:
            k_out = torch.empty((n_kv, Hkv, D), dtype=K.dtype, device=K.device)
        if v_out is None:
            v_out = torch.empty((n_kv, Hkv, D), dtype=V.dtype, device=V.device)
        cnt = _GatherCounts()
        _check(_lib().fcp_kv_gather_piece(self._h, rank, piece, K.data_ptr(), V.data_ptr(),
                                          k_out.data_ptr(), v_out.data_ptr(), Hkv,
                                          D * K.element_size() // 2, _stream_ptr(stream),
                                          C.byref(cnt)), "fcp_kv_gather_piece")
        return k_out, v_out, _struct_dict(cnt)

    def kv_scatter_add(self, rank, dk_r, dv_r, dK, dV, stream=None, piece=PIECE_FULL):
        """dK, dV (fp32 [C,Hkv,D]) += the rank's dk_r, dv_r (bf16 or fp32 [n_kv,Hkv,D], layout of
        the gathered KV).  Returns the counts dict (bytes a ReduceScatter would move)."""
        import torch
        for t in (dk_r, dv_r, dK, dV):
            assert t.is_cuda and t.is_contiguous()
        assert dK.dtype == torch.float32 and dV.dtype == torch.float32
        assert dk_r.dtype == dv_r.dtype and dk_r.dtype in (torch.bfloat16, torch.float32)
        Hkv, D = dK.shape[1], dK.shape[2]
        assert dk_r.shape[0] == self.rank_stats(rank, piece)["n_kv"] and dk_r.shape[1:] == dK.shape[1:]
        cnt = _GatherCounts()
        _check(_lib().fcp_kv_scatter_add_piece(self._h, rank, piece, dk_r.data_ptr(), dv_r.data_ptr(),
                                               0 if dk_r.dtype == torch.bfloat16 else 1,
                                               dK.data_ptr(), dV.data_ptr(), Hkv, D,
                                               _stream_ptr(stream), C.byref(cnt)),
               "fcp_kv_scatter_add_piece")
        return _struct_dict(cnt)

    def sched(self, rank, n_q_heads, n_kv_heads, head_dim, piece=PIECE_FULL):
        h = C.c_void_p()
        _check(_lib().fcp_sched_from_plan_piece(self._h, rank, piece, n_q_heads, n_kv_heads,
                                                head_dim, C.byref(h)), "fcp_sched_from_plan_piece")
        return Sched(h, n_q_heads, n_kv_heads, head_dim)


class Sched:
    """fcp_sched: tile schedule of one rank + its device workspace."""

    def __init__(self, handle, n_q_heads, n_kv_heads, head_dim):
        self._h = handle
        self.Hq, self.Hkv, self.D = n_q_heads, n_kv_heads, head_dim
        self.workspace = None

    @classmethod
    def create(cls, cu_seqlens_q, q_pos_off, shard_seg, cu_seqlens_k, n_q_heads, n_kv_heads,
               head_dim):
        cq, pp, sg, ck = _i32(cu_seqlens_q), _i32(q_pos_off), _i32(shard_seg), _i32(cu_seqlens_k)
        h = C.c_void_p()
        _check(_lib().fcp_sched_create(_p(cq), _p(pp), _p(sg), pp.size, _p(ck), ck.size - 1,
                                       n_q_heads, n_kv_heads, head_dim, C.byref(h)),
               "fcp_sched_create")
        return cls(h, n_q_heads, n_kv_heads, head_dim)

    def __del__(self):
        if getattr(self, "_h", None) and _LIB is not None:
            _LIB.fcp_sched_destroy(self._h)
            self._h = None

    def info(self):
        s = _SchedInfo()
        _check(_lib().fcp_sched_get_info(self._h, C.byref(s)), "fcp_sched_get_info")
        return _struct_dict(s)

    def lists(self):
        """Host work lists (fcp_sched_get_list) as int32 arrays: fwd [n,8], bwd [n,8], sub [n,4],
        fwd_cta / bwd_cta [n_cta+1]; field order in include/fcp.h."""
        out = {}
        for name, which, width in (("fwd", 0, 8), ("bwd", 1, 8), ("sub", 2, 4), ("fwd_cta", 3, 1),
                                   ("bwd_cta", 4, 1)):
            n = C.c_int64()
            _check(_lib().fcp_sched_get_list(self._h, which, None, 0, C.byref(n)),
                   "fcp_sched_get_list")
            a = np.zeros(max(n.value, 1), dtype=np.int32)
            _check(_lib().fcp_sched_get_list(self._h, which, _p(a), n.value, C.byref(n)),
                   "fcp_sched_get_list")
            a = a[:n.value]
            out[name] = a.reshape(-1, width) if width > 1 else a
        return out

    def workspace_size(self):
        n = C.c_size_t()
        _check(_lib().fcp_sched_workspace_size(self._h, C.byref(n)), "fcp_sched_workspace_size")
        return n.value

    def upload(self, device="cuda", stream=None, workspace=None):
        """Copy the item lists into the device workspace (allocated here unless the caller passes
        a uint8 tensor of at least workspace_size() bytes that it keeps alive and reuses; the
        caller then orders the copy stream against the kernels that still read the old lists)."""
        import torch
        if workspace is None:
            workspace = torch.empty(self.workspace_size(), dtype=torch.uint8, device=device)
        elif workspace.dtype != torch.uint8 or workspace.numel() < self.workspace_size() or \
                not workspace.is_cuda or not workspace.is_contiguous():
            raise ValueError("workspace must be a contiguous cuda uint8 tensor of >= %d bytes"
                             % self.workspace_size())
        self.workspace = workspace
        _check(_lib().fcp_sched_upload(self._h, self.workspace.data_ptr(), _stream_ptr(stream)),
               "fcp_sched_upload")
        return self

    def _args(self, q, k, v, o, lse, scale, stream, events=None, dkv_f32=False, dq_accum=None,
              dq_flags=0):
        if self.workspace is None:
            self.upload(q.device)
        ev0, ev1 = (None, None) if events is None else (_event_ptr(e) for e in events)
        return _AttnArgs(self._h, self.workspace.data_ptr(), q.data_ptr(), k.data_ptr(),
                         v.data_ptr(), o.data_ptr(), lse.data_ptr(), float(scale),
                         1 if dkv_f32 else 0, _stream_ptr(stream), ev0, ev1,
                         None if dq_accum is None else dq_accum.data_ptr(), dq_flags)

    def dq_accumulator(self, device="cuda"):
        """fp32 [Hq, n_q_pad, D] buffer for attn_bwd(dq_accum=...) over several KV pieces."""
        import torch
        return torch.empty((self.Hq, self.info()["n_q_pad"], self.D), dtype=torch.float32,
                           device=device)

    def attn_fwd(self, q, k, v, scale, o=None, lse=None, stream=None, events=None):
        """q [n_q,Hq,D], k,v [n_kv,Hkv,D] torch bf16 on the GPU -> (o bf16, lse f32 [Hq,n_q]).
        events = (start, stop) torch.cuda.Event pair recorded around the attention kernel."""
        import torch
        for t in (q, k, v):
            assert t.is_cuda and t.is_contiguous() and t.dtype == torch.bfloat16
        if o is None:
            o = torch.empty_like(q)
        if lse is None:
            lse = torch.empty((self.Hq, q.shape[0]), dtype=torch.float32, device=q.device)
        a = self._args(q, k, v, o, lse, scale, stream, events)
        _check(_lib().fcp_attn_fwd(C.byref(a)), "fcp_attn_fwd")
        return o, lse

    def attn_bwd(self, q, k, v, o, lse, do, scale, dq=None, dk=None, dv=None, stream=None,
                 events=None, dkv_dtype=None, dq_accum=None, dq_flags=0):
        """-> (dq bf16, dk, dv); dk, dv are bf16 unless dkv_dtype (or the given buffers) is f32.
        dq_accum / dq_flags (DQ_KEEP, DQ_NO_OUTPUT): dq accumulation over KV pieces, see
        fcp_attn_args in include/fcp.h; with DQ_NO_OUTPUT the returned dq is None."""
        import torch
        for t in (q, k, v, o, do):
            assert t.is_cuda and t.is_contiguous() and t.dtype == torch.bfloat16
        if dkv_dtype is None:
            dkv_dtype = dk.dtype if dk is not None else torch.bfloat16
        assert dkv_dtype in (torch.bfloat16, torch.float32)
        assert dq_accum is None or (dq_accum.is_cuda and dq_accum.dtype == torch.float32 and
                                    dq_accum.numel() == self.Hq * self.info()["n_q_pad"] * self.D)
        no_out = dq_accum is not None and (dq_flags & DQ_NO_OUTPUT)
        if not no_out:
            dq = torch.empty_like(q) if dq is None else dq
        dk = torch.empty_like(k, dtype=dkv_dtype) if dk is None else dk
        dv = torch.empty_like(v, dtype=dkv_dtype) if dv is None else dv
        assert dk.dtype == dkv_dtype and dv.dtype == dkv_dtype
        a = self._args(q, k, v, o, lse, scale, stream, events, dkv_dtype == torch.float32,
                       dq_accum, dq_flags)
        _check(_lib().fcp_attn_bwd(C.byref(a), do.data_ptr(), None if no_out else dq.data_ptr(),
                                   dk.data_ptr(), dv.data_ptr()), "fcp_attn_bwd")
        return (None if no_out else dq), dk, dv


    def attn_bwd_static(self, q, k, v, o, lse, do, scale, dq, dk, dv, stream=None):
        """fcp_attn_bwd_static: the backward on the library's own static device workspace, no
        upload() and no allocation anywhere (the outputs dq, dk, dv are the caller's tensors; dk,
        dv bf16 or f32).  FcpError(TOO_LARGE) when workspace_size() > STATIC_WORKSPACE_BYTES.
        Calls that overlap on the GPU race on the shared workspace (include/fcp.h)."""
        import torch
        for t in (q, k, v, o, do, dq):
            assert t.is_cuda and t.is_contiguous() and t.dtype == torch.bfloat16
        assert dk.dtype == dv.dtype and dk.dtype in (torch.bfloat16, torch.float32)
        assert dk.is_cuda and dv.is_cuda and dk.is_contiguous() and dv.is_contiguous()
        a = _AttnArgs(self._h, None, q.data_ptr(), k.data_ptr(), v.data_ptr(), o.data_ptr(),
                      lse.data_ptr(), float(scale), 1 if dk.dtype == torch.float32 else 0,
                      _stream_ptr(stream), None, None, None, 0)
        _check(_lib().fcp_attn_bwd_static(C.byref(a), do.data_ptr(), dq.data_ptr(), dk.data_ptr(),
                                          dv.data_ptr()), "fcp_attn_bwd_static")
        return dq, dk, dv


def kv_reduce_finish(dK, dV, dK_out=None, dV_out=None, stream=None):
    """fcp_kv_reduce_finish: the reduced fp32 dK, dV [C,Hkv,D] rounded to bf16 tensors."""
    import torch
    for t in (dK, dV):
        assert t.is_cuda and t.is_contiguous() and t.dtype == torch.float32
    dK_out = torch.empty_like(dK, dtype=torch.bfloat16) if dK_out is None else dK_out
    dV_out = torch.empty_like(dV, dtype=torch.bfloat16) if dV_out is None else dV_out
    assert dK_out.dtype == torch.bfloat16 and dV_out.dtype == torch.bfloat16
    assert dK.numel() == dV.numel() == dK_out.numel() == dV_out.numel()
    _check(_lib().fcp_kv_reduce_finish(dK.data_ptr(), dV.data_ptr(), dK_out.data_ptr(),
                                       dV_out.data_ptr(), dK.numel(), _stream_ptr(stream)),
           "fcp_kv_reduce_finish")
    return dK_out, dV_out


def merge(o_a, lse_a, o_b, lse_b, o_out=None, lse_out=None, stream=None):
    """fcp_merge on torch GPU tensors: o_* [rows,H,D] bf16 or f32, lse_* [H,rows] f32."""
    import torch
    assert o_a.is_cuda and o_a.is_contiguous() and o_b.is_contiguous()
    assert o_a.dtype == o_b.dtype and o_a.dtype in (torch.bfloat16, torch.float32)
    rows, H, D = o_a.shape
    o_out = torch.empty_like(o_a) if o_out is None else o_out
    lse_out = torch.empty_like(lse_a) if lse_out is None else lse_out
    _check(_lib().fcp_merge(o_a.data_ptr(), lse_a.data_ptr(), o_b.data_ptr(), lse_b.data_ptr(),
                            o_out.data_ptr(), lse_out.data_ptr(), rows, H, D,
                            0 if o_a.dtype == torch.bfloat16 else 1, _stream_ptr(stream)),
           "fcp_merge")
    return o_out, lse_out
