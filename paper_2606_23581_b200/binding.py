"""ctypes binding of libkamera (include/kamera.h): argument marshalling only.

Every function here has the name of the C entry point it calls.  torch is used for device memory and
streams - nothing is computed in Python.  If libkamera.so cannot be loaded this module raises: there is
no fallback path.
"""
import ctypes as C
import os

import torch

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))

KAM_OK, KAM_ERR_INVALID_ARG, KAM_ERR_NO_PAGES, KAM_ERR_UNSUPPORTED, KAM_ERR_STATE, KAM_ERR_CUDA = range(6)
KAM_MHA, KAM_GQA, KAM_MLA = 0, 1, 2
KAM_ROPE_HALF, KAM_ROPE_INTERLEAVED = 0, 1
KAM_PATCH_TARGET_FRAME, KAM_PATCH_CANONICAL_FRAME = 0, 1
KAM_FRONT, KAM_BACK = 0, 1
KAM_BF16, KAM_F32 = 0, 1
KAM_MAX_RANK, KAM_MAX_LAYERS = 64, 128
_STATUS = ["KAM_OK", "KAM_ERR_INVALID_ARG", "KAM_ERR_NO_PAGES", "KAM_ERR_UNSUPPORTED", "KAM_ERR_STATE", "KAM_ERR_CUDA"]

vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64


class kam_layout(C.Structure):
    _fields_ = [(n, i32) for n in ("kind", "n_layers", "n_q_heads", "n_kv_heads", "row_dim", "rope_off", "rope_dim",
                                    "has_v", "v_dim", "page_size", "rope_style", "elem_dtype", "factor_dtype")] + \
               [("rope_theta", C.c_double)]


class kam_pool(C.Structure):
    _fields_ = [("k_layers", vp), ("v_layers", vp), ("num_pages", i32)]


class kam_chunk(C.Structure):
    _fields_ = [("k_layers", vp), ("v_layers", vp), ("n_tokens", i32), ("p_base", i64)]


class kam_patch(C.Structure):
    _fields_ = [("Uk", vp), ("Wk", vp), ("Uv", vp), ("Wv", vp), ("u_token_stride", i64), ("u_head_stride", i64),
                ("rank_per_layer", C.POINTER(i32)), ("frame", i32)]


class kam_reloc_desc(C.Structure):
    _fields_ = [("block_table", vp), ("dst_token_start", i64), ("chunk", C.POINTER(kam_chunk)), ("p_target", i64),
                ("patch", C.POINTER(kam_patch)), ("rank", i32)]


class kam_patch_ref(C.Structure):
    _fields_ = [("Uk", vp), ("Wk", vp), ("Uv", vp), ("Wv", vp), ("u_token_stride", i64), ("u_head_stride", i64),
                ("rank", i32), ("frame", i32)]


class kam_stats(C.Structure):
    _fields_ = [(n, i64) for n in ("pages_free", "pages_total", "table_entries_written", "chunks_live",
                                    "kernels_launched", "device_errors", "generic_launches")]


# name -> (restype, argtypes): every symbol include/kamera.h declares
SIGNATURES = {
    "kam_create": (i32, [C.POINTER(kam_layout), C.POINTER(kam_pool), i32, i32, i32, C.POINTER(vp)]),
    "kam_destroy": (i32, [vp]),
    "kam_last_error": (C.c_char_p, [vp]),
    "kam_version": (C.c_char_p, []),
    "kam_set_option": (i32, [vp, C.c_char_p, i64]),
    "kam_relocate_patch": (i32, [vp, C.POINTER(kam_pool), vp, i64, C.POINTER(kam_chunk), i64, C.POINTER(kam_patch), i32,
                                 C.POINTER(kam_layout), vp]),
    "kam_relocate_patch_batch": (i32, [vp, C.POINTER(kam_pool), i32, C.POINTER(kam_reloc_desc), vp]),
    "kam_rotate_inplace": (i32, [vp, C.POINTER(kam_pool), vp, i64, i32, i64, vp]),
    "kam_relocate_patch_host": (i32, [vp, C.POINTER(kam_pool), vp, i64, i32, i64, i64, C.POINTER(vp), C.POINTER(vp),
                                      C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), i32, i32, vp]),
    "kam_form_patch": (i32, [vp, vp, vp, i32, i64, i32, i32, i32, vp, vp, vp, vp]),
    "kam_window_open": (i32, [vp, i32, i64]),
    "kam_window_pin": (i32, [vp, i32, i32]),
    "kam_window_close": (i32, [vp, i32]),
    "kam_admit": (i32, [vp, i32, i32, C.POINTER(kam_chunk), C.POINTER(kam_patch), i32, i32, C.POINTER(i32), vp]),
    "kam_evict": (i32, [vp, i32, i32, i32, vp]),
    "kam_slide": (i32, [vp, i32, i32, i32, C.POINTER(kam_chunk), C.POINTER(kam_patch), i32, i32, C.POINTER(i32), vp]),
    "kam_window_export": (i32, [vp, i32, C.POINTER(i32), i32, C.POINTER(i64), i64, C.POINTER(i32), C.POINTER(i64),
                                C.POINTER(i32), i32, C.POINTER(i32), C.POINTER(i32)]),
    "kam_get_stats": (i32, [vp, C.POINTER(kam_stats)]),
    "kam_paged_decode_merge": (i32, [vp, vp, C.POINTER(kam_pool), vp, i32, vp, vp, vp, i32, vp, i32, i32, C.c_float,
                                     vp, vp, vp]),
    "kam_paged_decode_plan": (i32, [vp, C.POINTER(kam_pool), vp, i32, vp, vp, vp, i32, i32, i32, vp]),
    "kam_paged_prefill_merge": (i32, [vp, vp, C.POINTER(kam_pool), vp, i32, vp, vp, vp, i32, i32, i32, i32, i32, C.c_float, vp, vp, vp]),
    "kam_decode_set_max_patch_rank": (i32, [vp, i32]),
    "kam_paged_decode_state": (i32, [vp, vp, C.POINTER(kam_pool), vp, i32, vp, vp, vp, i32, vp, i32, i32, C.c_float,
                                     vp, vp, vp]),
    "kam_lse_merge_states": (i32, [vp, i32, C.POINTER(vp), C.POINTER(vp), i32, vp, vp, vp]),
    "kam_window_plan": (i32, [vp, C.POINTER(i32), i32, vp]),
    "kam_window_decode": (i32, [vp, vp, C.POINTER(i32), i32, i32, C.c_float, vp, vp, vp]),
    "kam_paged_decode_merge_host": (i32, [vp, vp, C.POINTER(kam_pool), vp, i32, vp, vp, vp, i32, vp, i32, i32,
                                          C.c_float, vp, vp, vp]),
    "kam_paged_decode_merge_static": (i32, [C.POINTER(kam_layout), vp, C.POINTER(kam_pool), vp, i32, vp, vp, vp, i32, i32, i32,
                                            C.c_float, vp, vp, vp]),
}
KAM_STATIC_SCRATCH_BYTES = 16 << 20

_lib = None


def lib():
    """Load (building first if the sources are newer) libkamera.so.  Raises if that is impossible."""
    global _lib
    if _lib is None:
        path = _build.build()
        _lib = C.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(_lib, name)                     # AttributeError if the symbol is missing
            fn.restype, fn.argtypes = res, args
    return _lib


class KameraError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("%s: %s" % (_STATUS[status] if 0 <= status < len(_STATUS) else status, msg))
        self.status = status


def _check(status, ctx=None):
    if status != KAM_OK:
        msg = lib().kam_last_error(ctx)
        raise KameraError(status, msg.decode() if msg else "")


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return vp(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _ptr(t):
    return vp(t.data_ptr()) if t is not None else vp(None)


def _ptr_table(tensors, device):
    """Device int64 tensor holding the data_ptr of each per-layer tensor (a 'device array of device pointers')."""
    return torch.tensor([t.data_ptr() for t in tensors], dtype=torch.int64, device=device)


# ------------------------------------------------------------------------------------------------ argument holders
class Pool:
    """kam_pool over per-layer torch tensors [num_pages, P, H, D]; keeps the pointer tables alive."""

    def __init__(self, k_layers, v_layers=None):
        dev = k_layers[0].device
        self.k_layers, self.v_layers = list(k_layers), (list(v_layers) if v_layers is not None else None)
        self._kt = _ptr_table(self.k_layers, dev)
        self._vt = _ptr_table(self.v_layers, dev) if self.v_layers is not None else None
        self.c = kam_pool(_ptr(self._kt), _ptr(self._vt), k_layers[0].shape[0])


class Chunk:
    """kam_chunk over per-layer tensors [T, H, D]."""

    def __init__(self, k_layers, v_layers=None, p_base=0):
        dev = k_layers[0].device
        self.k_layers, self.v_layers = list(k_layers), (list(v_layers) if v_layers is not None else None)
        self._kt = _ptr_table(self.k_layers, dev)
        self._vt = _ptr_table(self.v_layers, dev) if self.v_layers is not None else None
        self.c = kam_chunk(_ptr(self._kt), _ptr(self._vt), k_layers[0].shape[0], int(p_base))


class Patch:
    """kam_patch over per-layer U [T, H, m] (or [T, m] shared by all heads) and W [H, m, D]."""

    def __init__(self, Uk, Wk, Uv=None, Wv=None, frame=KAM_PATCH_TARGET_FRAME, rank_per_layer=None):
        dev = Uk[0].device
        self.t = [list(x) if x is not None else None for x in (Uk, Wk, Uv, Wv)]
        self._tabs = [_ptr_table(x, dev) if x is not None else None for x in self.t]
        u = Uk[0]
        if u.dim() == 3:
            ts, hs = u.stride(0), u.stride(1)
        else:                                              # [T, m]: one U shared by all KV heads (paper's form)
            ts, hs = u.stride(0), 0
        self._rpl = (i32 * len(rank_per_layer))(*rank_per_layer) if rank_per_layer is not None else None
        self.rank = Wk[0].shape[1]
        self.c = kam_patch(*[_ptr(t) for t in self._tabs], ts, hs,
                           C.cast(self._rpl, C.POINTER(i32)) if self._rpl is not None else None, frame)


def make_layout(kind, n_layers, n_q_heads, n_kv_heads, row_dim, rope_off, rope_dim, has_v, page_size, rope_theta,
                rope_style=KAM_ROPE_HALF, elem_dtype=KAM_BF16, factor_dtype=KAM_BF16, v_dim=0):
    return kam_layout(kind, n_layers, n_q_heads, n_kv_heads, row_dim, rope_off, rope_dim, int(has_v), v_dim,
                      page_size, rope_style, elem_dtype, factor_dtype, float(rope_theta))


# ------------------------------------------------------------------------------------------------ the entry points
class Context:
    """Owns a kam_ctx*.  Methods carry the C names and do nothing but marshal."""

    def __init__(self, layout, pool=None, max_requests=0, max_chunks_per_request=0, max_pages_per_chunk=0):
        self.layout, self.pool = layout, pool
        h = vp()
        st = lib().kam_create(C.byref(layout), C.byref(pool.c) if pool is not None else None, max_requests,
                              max_chunks_per_request, max_pages_per_chunk, C.byref(h))
        _check(st, None)
        self.h = h

    def close(self):
        if getattr(self, "h", None) and _lib is not None:      # at interpreter shutdown the module globals may be gone already
            _lib.kam_destroy(self.h)
        self.h = None

    __del__ = close

    def kam_set_option(self, key, value):
        _check(lib().kam_set_option(self.h, key.encode(), int(value)), self.h)

    def kam_relocate_patch(self, block_table, dst_token_start, chunk, p_target, patch=None, rank=0, pool=None,
                           layout=None, stream=None):
        _check(lib().kam_relocate_patch(self.h, C.byref(pool.c) if pool else None, _ptr(block_table),
                                        int(dst_token_start), C.byref(chunk.c), int(p_target),
                                        C.byref(patch.c) if patch is not None else None, int(rank),
                                        C.byref(layout) if layout is not None else None, _stream_ptr(stream)), self.h)

    def kam_relocate_patch_batch(self, descs, pool=None, stream=None):
        """descs: list of (block_table, dst_token_start, chunk, p_target, patch or None, rank)."""
        arr = (kam_reloc_desc * len(descs))()
        for a, (bt, dst, ch, p, pa, r) in zip(arr, descs):
            a.block_table, a.dst_token_start, a.chunk, a.p_target = _ptr(bt), int(dst), C.pointer(ch.c), int(p)
            a.patch = C.pointer(pa.c) if pa is not None else None
            a.rank = int(r)
        _check(lib().kam_relocate_patch_batch(self.h, C.byref(pool.c) if pool else None, len(descs), arr,
                                              _stream_ptr(stream)), self.h)

    def kam_rotate_inplace(self, block_table, token_start, n_tokens, delta, pool=None, stream=None):
        _check(lib().kam_rotate_inplace(self.h, C.byref(pool.c) if pool else None, _ptr(block_table),
                                        int(token_start), int(n_tokens), int(delta), _stream_ptr(stream)), self.h)

    def kam_relocate_patch_host(self, block_table, dst_token_start, n_tokens, p_base, p_target, k_host, v_host,
                                Uk_host, Wk_host, Uv_host, Wv_host, rank, frame=KAM_PATCH_TARGET_FRAME, pool=None,
                                stream=None):
        def tab(ts):
            return (vp * len(ts))(*[t.data_ptr() for t in ts]) if ts is not None else None
        _check(lib().kam_relocate_patch_host(self.h, C.byref(pool.c) if pool else None, _ptr(block_table),
                                             int(dst_token_start), int(n_tokens), int(p_base), int(p_target),
                                             tab(k_host), tab(v_host), tab(Uk_host), tab(Wk_host), tab(Uv_host),
                                             tab(Wv_host), int(rank), int(frame), _stream_ptr(stream)), self.h)

    def kam_form_patch(self, kv_cond_layers, kv_solo_layers, delta, is_key, rank, n_iter=0, sigma=None, stream=None):
        """kv_*_layers: lists of per-layer device tensors [T, H, D].  Returns (U list [T, H, rank], W list [H, rank, D])."""
        dev, T = kv_cond_layers[0].device, kv_cond_layers[0].shape[0]
        H, D = self.layout.n_kv_heads, self.layout.row_dim
        U = [torch.empty((T, H, rank), dtype=torch.bfloat16, device=dev) for _ in kv_cond_layers]
        W = [torch.empty((H, rank, D), dtype=torch.bfloat16, device=dev) for _ in kv_cond_layers]
        tabs = [_ptr_table(x, dev) for x in (kv_cond_layers, kv_solo_layers, U, W)]
        _check(lib().kam_form_patch(self.h, _ptr(tabs[0]), _ptr(tabs[1]), T, int(delta), int(is_key), int(rank), int(n_iter),
                                    _ptr(tabs[2]), _ptr(tabs[3]), _ptr(sigma), _stream_ptr(stream)), self.h)
        torch.cuda.current_stream().synchronize() if stream is None else None      # the pointer tables must outlive the launch
        return U, W

    # ---- window store
    def kam_window_open(self, req, window_base=0):
        _check(lib().kam_window_open(self.h, req, int(window_base)), self.h)

    def kam_window_pin(self, req, n_front_chunks):
        _check(lib().kam_window_pin(self.h, req, n_front_chunks), self.h)

    def kam_window_close(self, req):
        _check(lib().kam_window_close(self.h, req), self.h)

    def kam_admit(self, req, end, chunk, patch=None, rank=0, materialize=1, stream=None):
        handle = i32(-1)
        sp = _stream_ptr(stream) if torch.cuda.is_available() else vp(None)
        _check(lib().kam_admit(self.h, req, end, C.byref(chunk.c if hasattr(chunk, "c") else chunk),
                               C.byref(patch.c) if patch is not None else None, int(rank), int(materialize),
                               C.byref(handle), sp), self.h)
        return handle.value

    def kam_evict(self, req, end, materialize=1, stream=None):
        sp = _stream_ptr(stream) if torch.cuda.is_available() else vp(None)
        _check(lib().kam_evict(self.h, req, end, int(materialize), sp), self.h)

    def kam_slide(self, req, evict_end, admit_end, chunk, patch=None, rank=0, materialize=1, stream=None):
        handle = i32(-1)
        sp = _stream_ptr(stream) if torch.cuda.is_available() else vp(None)
        _check(lib().kam_slide(self.h, req, evict_end, admit_end, C.byref(chunk.c if hasattr(chunk, "c") else chunk),
                               C.byref(patch.c) if patch is not None else None, int(rank), int(materialize),
                               C.byref(handle), sp), self.h)
        return handle.value

    def kam_window_export(self, req):
        n_pages, n_chunks = i32(), i32()
        _check(lib().kam_window_export(self.h, req, None, 0, None, 0, None, None, None, 0, C.byref(n_pages),
                                       C.byref(n_chunks)), self.h)
        P = self.layout.page_size
        bt = (i32 * max(1, n_pages.value))()
        sm = (i64 * max(1, n_pages.value * P))()
        st = (i32 * (n_chunks.value + 1))()
        of = (i64 * (n_chunks.value + 1))()
        hd = (i32 * (n_chunks.value + 1))()
        _check(lib().kam_window_export(self.h, req, bt, n_pages.value, sm, n_pages.value * P, st, of, hd,
                                       n_chunks.value + 1, C.byref(n_pages), C.byref(n_chunks)), self.h)
        nc, npg = n_chunks.value, n_pages.value
        return {"block_table": list(bt[:npg]), "slot_mapping": list(sm[:npg * P]), "chunk_starts": list(st[:nc + 1]),
                "chunk_offsets": list(of[:nc]), "handles": list(hd[:nc])}

    def kam_get_stats(self):
        s = kam_stats()
        _check(lib().kam_get_stats(self.h, C.byref(s)), self.h)
        return {n: getattr(s, n) for n, _ in kam_stats._fields_}

    # ---- decode
    def kam_paged_decode_merge(self, q, block_tables, chunk_starts, chunk_offsets, n_chunks, layer, sm_scale, out,
                               lse, patches=None, pool=None, stream=None):
        batch, max_pages = block_tables.shape
        max_chunks = chunk_starts.shape[1] - 1
        _check(lib().kam_paged_decode_merge(self.h, _ptr(q), C.byref(pool.c) if pool else None, _ptr(block_tables),
                                            max_pages, _ptr(chunk_starts), _ptr(chunk_offsets), _ptr(n_chunks),
                                            max_chunks, _ptr(patches), int(layer), batch, float(sm_scale), _ptr(out),
                                            _ptr(lse), _stream_ptr(stream)), self.h)

    def kam_paged_decode_plan(self, block_tables, chunk_starts, chunk_offsets, n_chunks, has_patches=False, pool=None,
                              stream=None):
        """Pins the plan of these metadata arrays (None block_tables releases it)."""
        if block_tables is None:
            _check(lib().kam_paged_decode_plan(self.h, None, None, 0, None, None, None, 0, 0, 0, _stream_ptr(stream)), self.h)
            return
        batch, max_pages = block_tables.shape
        max_chunks = chunk_starts.shape[1] - 1
        _check(lib().kam_paged_decode_plan(self.h, C.byref(pool.c) if pool else None, _ptr(block_tables), max_pages,
                                           _ptr(chunk_starts), _ptr(chunk_offsets), _ptr(n_chunks), max_chunks,
                                           int(bool(has_patches)), batch, _stream_ptr(stream)), self.h)

    def kam_paged_prefill_merge(self, q, block_tables, chunk_starts, chunk_offsets, n_chunks, layer, causal, sm_scale, out, lse,
                                pool=None, stream=None):
        """q, out: [batch, n_q_tokens, Hq, D] bf16; lse [batch, n_q_tokens, Hq] f32."""
        batch, max_pages = block_tables.shape
        max_chunks = chunk_starts.shape[1] - 1
        _check(lib().kam_paged_prefill_merge(self.h, _ptr(q), C.byref(pool.c) if pool else None, _ptr(block_tables), max_pages,
                                             _ptr(chunk_starts), _ptr(chunk_offsets), _ptr(n_chunks), max_chunks, int(layer), batch,
                                             int(q.shape[1]), int(bool(causal)), float(sm_scale), _ptr(out), _ptr(lse),
                                             _stream_ptr(stream)), self.h)

    def kam_paged_decode_state(self, q, block_tables, chunk_starts, chunk_offsets, n_chunks, layer, sm_scale, o_state,
                               lse_state, patches=None, pool=None, stream=None):
        batch, max_pages = block_tables.shape
        max_chunks = chunk_starts.shape[1] - 1
        _check(lib().kam_paged_decode_state(self.h, _ptr(q), C.byref(pool.c) if pool else None, _ptr(block_tables),
                                            max_pages, _ptr(chunk_starts), _ptr(chunk_offsets), _ptr(n_chunks),
                                            max_chunks, _ptr(patches), int(layer), batch, float(sm_scale),
                                            _ptr(o_state), _ptr(lse_state), _stream_ptr(stream)), self.h)

    def kam_lse_merge_states(self, o_states, lse_states, batch, out, lse, stream=None):
        """o_states / lse_states: lists of device tensors (one per part), or data pointers (peer memory)."""
        ptr = lambda t: t.data_ptr() if hasattr(t, "data_ptr") else int(t)
        n = len(o_states)
        oa = (vp * n)(*[ptr(t) for t in o_states])
        la = (vp * n)(*[ptr(t) for t in lse_states])
        _check(lib().kam_lse_merge_states(self.h, n, oa, la, int(batch), _ptr(out), _ptr(lse), _stream_ptr(stream)), self.h)

    def kam_decode_set_max_patch_rank(self, max_rank):
        _check(lib().kam_decode_set_max_patch_rank(self.h, int(max_rank)), self.h)

    def kam_window_plan(self, req_ids, stream=None):
        ids = (i32 * len(req_ids))(*req_ids)
        _check(lib().kam_window_plan(self.h, ids, len(req_ids), _stream_ptr(stream)), self.h)

    def kam_window_decode(self, q, req_ids, layer, sm_scale, out, lse, stream=None):
        ids = (i32 * len(req_ids))(*req_ids)
        _check(lib().kam_window_decode(self.h, _ptr(q), ids, len(req_ids), int(layer), float(sm_scale), _ptr(out),
                                       _ptr(lse), _stream_ptr(stream)), self.h)

    def kam_paged_decode_merge_host(self, q_host, block_tables, chunk_starts, chunk_offsets, n_chunks, layer, sm_scale,
                                    out_host, lse_host, patches=None, pool=None, stream=None):
        batch, max_pages = block_tables.shape
        max_chunks = chunk_starts.shape[1] - 1
        _check(lib().kam_paged_decode_merge_host(self.h, _ptr(q_host), C.byref(pool.c) if pool else None,
                                                 _ptr(block_tables), max_pages, _ptr(chunk_starts), _ptr(chunk_offsets),
                                                 _ptr(n_chunks), max_chunks, _ptr(patches), int(layer), batch,
                                                 float(sm_scale), _ptr(out_host), _ptr(lse_host), _stream_ptr(stream)),
               self.h)


def kam_paged_decode_merge_static(layout, q, pool, block_tables, chunk_starts, chunk_offsets, n_chunks, layer, sm_scale, out, lse,
                                  stream=None):
    """The fused decode without a context and without any device allocation inside the library (kamera.h): for hosts that have
    given all their HBM to an allocator of their own, or that may not pay cudaMalloc's device-wide synchronisation.  Scratch is
    the library's static 16 MiB device array - shared by every caller on the device, so calls must be ordered on one stream."""
    batch, max_pages = block_tables.shape
    max_chunks = chunk_starts.shape[1] - 1
    _check(lib().kam_paged_decode_merge_static(C.byref(layout), _ptr(q), C.byref(pool.c), _ptr(block_tables), max_pages,
                                               _ptr(chunk_starts), _ptr(chunk_offsets), _ptr(n_chunks), max_chunks, int(layer),
                                               batch, float(sm_scale), _ptr(out), _ptr(lse), _stream_ptr(stream)), None)


def patch_refs(refs, device, max_chunks=None):
    """Device array of kam_patch_ref [batch][max_chunks] from nested lists of (Uk, Wk, Uv, Wv, rank[, frame]) or None."""
    batch = len(refs)
    max_chunks = max_chunks if max_chunks is not None else max(len(r) for r in refs)
    arr = (kam_patch_ref * (batch * max_chunks))()
    keep = []
    for b, row in enumerate(refs):
        for c, ref in enumerate(row):
            if ref is None:
                continue
            Uk, Wk, Uv, Wv, rank = ref[:5]
            a = arr[b * max_chunks + c]
            a.Uk, a.Wk, a.Uv, a.Wv = _ptr(Uk), _ptr(Wk), _ptr(Uv), _ptr(Wv)
            a.u_token_stride, a.u_head_stride = (Uk.stride(0), Uk.stride(1)) if Uk.dim() == 3 else (Uk.stride(0), 0)
            a.rank = int(rank)
            a.frame = int(ref[5]) if len(ref) > 5 else KAM_PATCH_TARGET_FRAME
            keep.append(ref)
    raw = torch.frombuffer(bytearray(bytes(arr)), dtype=torch.uint8).to(device)
    raw._keep = keep
    return raw
