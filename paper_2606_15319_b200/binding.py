"""ctypes binding of libslack.so (include/slack.h) — argument marshalling only.

Every step of the hot path (append, plan, attention, combine) runs inside the library; this module converts torch
tensors / StreamSpec-like objects to the plain pointers and structs of the C ABI and raises on any non-OK status.
It never falls back to anything: a missing library raises ImportError-like RuntimeError at load time.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_PKG_DIR = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG_DIR, "libslack.so")

SLACK_OK, SLACK_EINVAL, SLACK_EUNSUPPORTED, SLACK_ENOMEM, SLACK_ECUDA, SLACK_ESTALE_PLAN = range(6)
STATUS_NAMES = ["SLACK_OK", "SLACK_EINVAL", "SLACK_EUNSUPPORTED", "SLACK_ENOMEM", "SLACK_ECUDA", "SLACK_ESTALE_PLAN"]
SLACK_BF16, SLACK_F32, SLACK_FP8_E4M3 = 0, 1, 2
DTYPES = {"bf16": SLACK_BF16, "f32": SLACK_F32, "fp8": SLACK_FP8_E4M3}


class SlackError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES[status] if 0 <= status < 6 else status}: {message}")
        self.status = status


class CPool(C.Structure):
    _fields_ = [("k_pool", C.c_void_p), ("v_pool", C.c_void_p), ("n_pages", C.c_int32), ("n_heads", C.c_int32),
                ("head_dim", C.c_int32), ("page_size", C.c_int32), ("dtype", C.c_int32), ("reserved", C.c_int32),
                ("k_scale", C.c_void_p), ("v_scale", C.c_void_p)]


class CStream(C.Structure):
    _fields_ = [("q_len", C.c_int32), ("cache_len", C.c_int32), ("base", C.c_int32), ("window", C.c_int32),
                ("sink_len", C.c_int32), ("gap_slots", C.c_int32), ("n_table_pages", C.c_int32), ("reserved", C.c_int32),
                ("page_table", C.POINTER(C.c_int32))]


class CPlanOpts(C.Structure):
    _fields_ = [("sm_count", C.c_int32), ("force_splits", C.c_int32), ("force_simt", C.c_int32), ("cta_pairs", C.c_int32)]


class CWorkItem(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("stream", "head", "q_row0", "q_rows", "kv_tile_begin", "kv_tile_end",
                                         "pos_lo", "pos_hi", "sink_tiles", "sink_pos_hi", "partial_slot", "cta", "dual")]


# every symbol include/slack.h declares: name -> (restype, argtypes)
_VP = C.c_void_p
SYMBOLS = {
    "slack_abi_version": (C.c_int32, []),
    "slack_create": (C.c_int, [C.POINTER(_VP), C.c_int]),
    "slack_destroy": (None, [_VP]),
    "slack_last_error": (C.c_char_p, [_VP]),
    "slack_last_launch_count": (C.c_int32, [_VP]),
    "slack_kv_append": (C.c_int, [_VP, C.POINTER(CPool), C.c_int32, C.POINTER(CStream), _VP, _VP, _VP]),
    "slack_kv_append_planned": (C.c_int, [_VP, _VP, C.POINTER(CPool), _VP, _VP, _VP]),
    "slack_plan": (C.c_int, [_VP, C.POINTER(CPool), C.c_int32, C.POINTER(CStream), C.POINTER(CPlanOpts), C.POINTER(_VP)]),
    "slack_plan_destroy": (None, [_VP]),
    "slack_plan_workspace_bytes": (C.c_size_t, [_VP]),
    "slack_plan_num_items": (C.c_int32, [_VP]),
    "slack_plan_num_partial_slots": (C.c_int32, [_VP]),
    "slack_plan_kernel_kind": (C.c_int32, [_VP]),
    "slack_plan_get_items": (C.c_int32, [_VP, C.POINTER(CWorkItem), C.c_int32]),
    "slack_chunk_attention": (C.c_int, [_VP, _VP, C.POINTER(CPool), _VP, _VP, _VP, C.c_float, _VP, C.c_size_t, _VP]),
    "slack_chunk_attention_static": (C.c_int, [_VP, _VP, C.POINTER(CPool), _VP, _VP, _VP, C.c_float, _VP]),
    "slack_static_workspace_init": (C.c_int, [_VP, C.POINTER(C.c_size_t)]),
    "slack_chunk_attention_sparse": (C.c_int, [_VP, _VP, C.POINTER(CPool), _VP, _VP, _VP, C.c_float, _VP, C.c_int32, _VP,
                                              C.c_size_t, _VP]),
    "slack_plan_sparse_workspace_bytes": (C.c_size_t, [_VP]),
    "slack_plan_mask_rows": (C.c_int32, [_VP]),
    "slack_plan_mask_min_words": (C.c_int32, [_VP]),
    "slack_kv_transfer": (C.c_int, [_VP, C.c_int32, C.POINTER(CPool), C.POINTER(CPool), C.c_int32, C.POINTER(C.c_int32),
                                   C.POINTER(C.c_int32), C.c_int32, C.c_int32, _VP, C.POINTER(_VP)]),
    "slack_profile_enable": (C.c_int, [_VP, C.c_int32]),
    "slack_profile_read": (C.c_int, [_VP, C.c_int32, C.POINTER(C.c_double), C.c_int32, C.POINTER(C.c_int32)]),
    "slack_cache_create": (C.c_int, [C.c_int32, C.c_int32, C.c_int32, C.POINTER(_VP)]),
    "slack_cache_destroy": (None, [_VP]),
    "slack_cache_open": (C.c_int, [_VP, C.c_int32, C.c_int32, C.POINTER(C.c_int32)]),
    "slack_cache_begin_chunk": (C.c_int, [_VP, C.c_int32, C.c_int32, C.POINTER(CStream)]),
    "slack_cache_commit": (C.c_int, [_VP, C.c_int32]),
    "slack_cache_close": (C.c_int, [_VP, C.c_int32]),
    "slack_cache_free_pages": (C.c_int32, [_VP]),
    "slack_cache_stream_pages": (C.c_int32, [_VP, C.c_int32]),
    "slack_cache_last_error": (C.c_char_p, [_VP]),
}
# include/slack_diag.h: only a library built with -DSLACK_DIAGNOSTICS exports these
DIAG_SYMBOLS = {"slack_debug_set": (C.c_int, [_VP, C.c_int32, _VP])}
PROF_ATTENTION, PROF_APPEND, PROF_COMBINE = 1, 2, 4
TRIM_PAGES, TRIM_TOKENS = 0, 1

_lib = None


def load() -> C.CDLL:
    """dlopen libslack.so and type its symbols; raises if the library has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_15319_b200.build` "
                               "(there is no fallback path)")
        lib = C.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        for name, (res, args) in DIAG_SYMBOLS.items():
            if hasattr(lib, name):
                fn = getattr(lib, name)
                fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def _stream_array(streams: Sequence):
    """slack_stream[] from StreamSpec-like objects (q_len, cache_len, base, window, sink_len, gap_slots, page_table)."""
    arr = (CStream * max(len(streams), 1))()
    keep = []
    for i, s in enumerate(streams):
        table = np.ascontiguousarray(s.page_table, dtype=np.int32)
        keep.append(table)
        arr[i] = CStream(int(s.q_len), int(s.cache_len), int(s.base), int(s.window), int(getattr(s, "sink_len", 0)),
                         int(getattr(s, "gap_slots", 0)), int(table.size), 0, table.ctypes.data_as(C.POINTER(C.c_int32)))
    return arr, keep


def _ptr(t) -> Optional[int]:
    if t is None:
        return None
    if isinstance(t, int):
        return t
    return t.data_ptr()


def _cuda_stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        if torch.cuda.is_available():
            return torch.cuda.current_stream().cuda_stream or None
        return None
    if isinstance(stream, int):
        return stream or None
    return stream.cuda_stream or None


class Pool:
    """One layer's K/V pool: torch tensors [n_pages, H, P, D] (bf16 or f32), caller-owned.  dtype "fp8": uint8 tensors of
    e4m3 codes plus k_scale / v_scale, fp32 [n_pages, H, P // 128] (include/slack.h slack_dtype)."""

    def __init__(self, k_pool, v_pool, n_pages: int, n_heads: int, head_dim: int, page_size: int, dtype: str,
                 k_scale=None, v_scale=None):
        self.k_pool, self.v_pool, self.k_scale, self.v_scale = k_pool, v_pool, k_scale, v_scale
        self.c = CPool(_ptr(k_pool), _ptr(v_pool), n_pages, n_heads, head_dim, page_size, DTYPES[dtype], 0,
                       _ptr(k_scale), _ptr(v_scale))

    @classmethod
    def shape_only(cls, n_pages, n_heads, head_dim, page_size, dtype):
        return cls(None, None, n_pages, n_heads, head_dim, page_size, dtype)


class Plan:
    def __init__(self, ctx: "Context", handle: int):
        self.ctx, self.handle = ctx, handle

    def close(self):
        if self.handle:
            load().slack_plan_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def workspace_bytes(self) -> int:
        return int(load().slack_plan_workspace_bytes(self.handle))

    @property
    def sparse_workspace_bytes(self) -> int:
        return int(load().slack_plan_sparse_workspace_bytes(self.handle))

    @property
    def mask_rows(self) -> int:
        return int(load().slack_plan_mask_rows(self.handle))

    @property
    def mask_min_words(self) -> int:
        return int(load().slack_plan_mask_min_words(self.handle))

    @property
    def num_items(self) -> int:
        return int(load().slack_plan_num_items(self.handle))

    @property
    def num_partial_slots(self) -> int:
        return int(load().slack_plan_num_partial_slots(self.handle))

    @property
    def kernel_kind(self) -> int:
        return int(load().slack_plan_kernel_kind(self.handle))

    def items(self):
        n = self.num_items
        buf = (CWorkItem * max(n, 1))()
        got = load().slack_plan_get_items(self.handle, buf, n)
        names = [f[0] for f in CWorkItem._fields_]
        return [{k: int(getattr(buf[i], k)) for k in names} for i in range(got)]


class Context:
    """slack_ctx wrapper. device=-1 gives a host-only context (planning / inspection only)."""

    def __init__(self, device: int = 0):
        self.lib = load()
        h = _VP()
        st = self.lib.slack_create(C.byref(h), device)
        if st != SLACK_OK:
            raise SlackError(st, f"slack_create(device={device}) failed")
        self.handle = h.value
        self.device = device

    def close(self):
        if getattr(self, "handle", None):
            self.lib.slack_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st: int):
        if st != SLACK_OK:
            raise SlackError(st, self.lib.slack_last_error(self.handle).decode())

    @property
    def last_launch_count(self) -> int:
        return int(self.lib.slack_last_launch_count(self.handle))

    # --- the three calls of the boundary, same names as the C ABI ---------------------------------------------------
    def slack_plan(self, pool: Pool, streams: Sequence, sm_count: int = 0, force_splits: int = 0,
                   force_simt: int = 0, cta_pairs: int = 0) -> Plan:
        arr, keep = _stream_array(streams)
        opts = CPlanOpts(sm_count, force_splits, force_simt, cta_pairs)
        h = _VP()
        self._check(self.lib.slack_plan(self.handle, C.byref(pool.c), len(streams), arr, C.byref(opts), C.byref(h)))
        del keep
        return Plan(self, h.value)

    def slack_kv_append(self, pool: Pool, streams: Sequence, k_new, v_new, stream=None) -> None:
        arr, keep = _stream_array(streams)
        self._check(self.lib.slack_kv_append(self.handle, C.byref(pool.c), len(streams), arr, _ptr(k_new), _ptr(v_new),
                                             _cuda_stream(stream)))
        del keep

    def slack_kv_append_planned(self, plan: Plan, pool: Pool, k_new, v_new, stream=None) -> None:
        self._check(self.lib.slack_kv_append_planned(self.handle, plan.handle, C.byref(pool.c), _ptr(k_new), _ptr(v_new),
                                                     _cuda_stream(stream)))

    def slack_chunk_attention(self, plan: Plan, pool: Pool, q, out, scale: float, lse=None, workspace=None,
                              stream=None) -> None:
        ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
        self._check(self.lib.slack_chunk_attention(self.handle, plan.handle, C.byref(pool.c), _ptr(q), _ptr(out), _ptr(lse),
                                                   C.c_float(scale), _ptr(workspace), ws_bytes, _cuda_stream(stream)))

    def slack_static_workspace_init(self) -> int:
        """Resolves the static workspace of this context's device; returns its size (the limit) in bytes."""
        n = C.c_size_t(0)
        self._check(self.lib.slack_static_workspace_init(self.handle, C.byref(n)))
        return int(n.value)

    def slack_chunk_attention_static(self, plan: Plan, pool: Pool, q, out, scale: float, lse=None, stream=None) -> None:
        """slack_chunk_attention with the library's static workspace (no allocation; include/slack.h for the limit)."""
        self._check(self.lib.slack_chunk_attention_static(self.handle, plan.handle, C.byref(pool.c), _ptr(q), _ptr(out),
                                                          _ptr(lse), C.c_float(scale), _cuda_stream(stream)))

    def slack_chunk_attention_sparse(self, plan: Plan, pool: Pool, q, out, scale: float, block_mask, lse=None,
                                     workspace=None, stream=None) -> None:
        """block_mask: int32/uint32 device tensor [plan.mask_rows][n_heads][mask_words] (include/slack.h)."""
        ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
        self._check(self.lib.slack_chunk_attention_sparse(self.handle, plan.handle, C.byref(pool.c), _ptr(q), _ptr(out),
                                                          _ptr(lse), C.c_float(scale), _ptr(block_mask),
                                                          int(block_mask.shape[-1]), _ptr(workspace), ws_bytes,
                                                          _cuda_stream(stream)))

    def slack_kv_transfer(self, src_pools: Sequence[Pool], dst_pools: Sequence[Pool], src_page_ids, dst_page_ids,
                          head_begin: int, head_end: int, stream=None, layer_done_events=None) -> None:
        """Layer-major page transfer (include/slack.h).  layer_done_events: optional list of torch.cuda.Event (one per
        layer, already created with .record()-able handles) recorded after each layer's copy."""
        n_layers = len(src_pools)
        assert len(dst_pools) == n_layers
        sp = (CPool * max(n_layers, 1))(*[p.c for p in src_pools])
        dp = (CPool * max(n_layers, 1))(*[p.c for p in dst_pools])
        a = np.ascontiguousarray(src_page_ids, dtype=np.int32)
        b = np.ascontiguousarray(dst_page_ids, dtype=np.int32)
        assert a.size == b.size
        ev = None
        if layer_done_events is not None:
            ev = (_VP * n_layers)(*[int(e.cuda_event) for e in layer_done_events])
        self._check(self.lib.slack_kv_transfer(self.handle, n_layers, sp, dp, int(a.size),
                                               a.ctypes.data_as(C.POINTER(C.c_int32)), b.ctypes.data_as(C.POINTER(C.c_int32)),
                                               int(head_begin), int(head_end), _cuda_stream(stream), ev))

    # --- measurement ---------------------------------------------------------------------------------------------------
    def profile_enable(self, kinds: int) -> None:
        """kinds: OR of PROF_ATTENTION / PROF_APPEND / PROF_COMBINE (0 = off); see include/slack.h."""
        self._check(self.lib.slack_profile_enable(self.handle, int(kinds)))

    def profile_read(self, kind: int, capacity: int = 1 << 16):
        """Per-launch durations (ms, launch order) of one kernel kind since the last read."""
        buf = (C.c_double * capacity)()
        n = C.c_int32(0)
        self._check(self.lib.slack_profile_read(self.handle, int(kind), buf, capacity, C.byref(n)))
        return [float(buf[i]) for i in range(min(int(n.value), capacity))]

    # --- diagnostics (library built with SLACK_DIAGNOSTICS=1 only; include/slack_diag.h) ------------------------------
    def debug_set(self, key: int, tensor) -> None:
        if not hasattr(self.lib, "slack_debug_set"):
            raise RuntimeError("libslack.so was built without -DSLACK_DIAGNOSTICS")
        self._check(self.lib.slack_debug_set(self.handle, int(key), _ptr(tensor)))


class Cache:
    """slack_cache_t wrapper: page bookkeeping of one pool shape (A0 / A5, host only).  begin_chunk returns a descriptor
    object with the StreamSpec fields (page_table copied out as a numpy array)."""

    class Desc:
        def __init__(self, c: "CStream"):
            self.q_len, self.cache_len, self.base, self.window = c.q_len, c.cache_len, c.base, c.window
            self.sink_len, self.gap_slots = c.sink_len, c.gap_slots
            self.page_table = np.ctypeslib.as_array(c.page_table, shape=(c.n_table_pages,)).copy() if c.n_table_pages else \
                np.zeros(0, dtype=np.int32)

        @property
        def n(self) -> int:
            return self.cache_len + self.q_len

    def __init__(self, n_pages: int, page_size: int, trim_policy: int = TRIM_PAGES):
        self.lib = load()
        h = _VP()
        st = self.lib.slack_cache_create(n_pages, page_size, trim_policy, C.byref(h))
        if st != SLACK_OK:
            raise SlackError(st, "slack_cache_create failed")
        self.handle = h.value

    def close(self):
        if getattr(self, "handle", None):
            self.lib.slack_cache_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st: int):
        if st != SLACK_OK:
            raise SlackError(st, self.lib.slack_cache_last_error(self.handle).decode())

    def open(self, window: int = 0, sink_len: int = 0) -> int:
        sid = C.c_int32(-1)
        self._check(self.lib.slack_cache_open(self.handle, window, sink_len, C.byref(sid)))
        return int(sid.value)

    def begin_chunk(self, stream_id: int, q_len: int) -> "Cache.Desc":
        c = CStream()
        self._check(self.lib.slack_cache_begin_chunk(self.handle, stream_id, q_len, C.byref(c)))
        return Cache.Desc(c)

    def commit(self, stream_id: int) -> None:
        self._check(self.lib.slack_cache_commit(self.handle, stream_id))

    def close_stream(self, stream_id: int) -> None:
        self._check(self.lib.slack_cache_close(self.handle, stream_id))

    @property
    def free_pages(self) -> int:
        return int(self.lib.slack_cache_free_pages(self.handle))

    def stream_pages(self, stream_id: int) -> int:
        return int(self.lib.slack_cache_stream_pages(self.handle, stream_id))


# ---------------------------------------------------------------------------------------------------------------------
# storage helpers (numpy bit patterns <-> torch tensors); no arithmetic
# ---------------------------------------------------------------------------------------------------------------------

def to_torch(arr: np.ndarray, dtype: str, device="cpu", pin: bool = False):
    """numpy storage array (uint16 bf16 bit patterns, or float32) -> torch tensor of the same bits."""
    import torch
    a = np.ascontiguousarray(arr)
    t = torch.from_numpy(a.view(np.int16)).view(torch.bfloat16) if dtype == "bf16" else torch.from_numpy(a)
    if pin:
        t = t.pin_memory()
    return t.to(device) if str(device) != "cpu" else t


def to_numpy(t, dtype: str) -> np.ndarray:
    """torch tensor -> numpy storage array (uint16 bit patterns for bf16)."""
    import torch
    t = t.detach().cpu().contiguous()
    if dtype == "bf16":
        return t.view(torch.int16).numpy().view(np.uint16)
    return t.numpy()
