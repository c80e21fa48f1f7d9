"""Thin ctypes binding of libkvtier.so (include/kvtier.h): same names, argument marshalling only.

Every step of the path (page-id staging, address generation, pack / unpack / re-page, host-tier
offload / reload) runs inside the library's sm_100a kernels and copy-engine calls; nothing here
touches transfer data.  PyTorch tensors are accepted only as a source of device pointers and
stream handles.  Loading fails loudly when the library has not been built: there is no
fallback path.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libkvtier.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build it with `python -c 'import __graft_entry__ as g; g.build()'` "
        "(nvcc, sm_100a).  kvtier has no CPU or PyTorch fallback."
    )
_lib = ctypes.CDLL(LIB_PATH)

# ---- enums (include/kvtier.h) ------------------------------------------------------------------
KV_OK = 0
KV_ERR_NULL, KV_ERR_SIZE, KV_ERR_PAGE_RANGE, KV_ERR_DUP_PAGE, KV_ERR_LAYOUT = -1, -2, -3, -4, -5
KV_ERR_ALIGN, KV_ERR_CUDA, KV_ERR_HOST_MEM, KV_ERR_DESC, KV_ERR_NO_DEVICE = -6, -7, -8, -9, -10
KV_ERR_CAPTURE = -11
KV_ERR_STATIC_LIMIT = -12
KV_STATIC_MAX_PAGES, KV_STATIC_MAX_SLABS = 65536, 1024
KV_STATIC_TABLE_BYTES = 256 + KV_STATIC_MAX_SLABS * 8 + KV_STATIC_MAX_PAGES * 4
KV_LAYOUT_PAGE_FIRST, KV_LAYOUT_LAYER_FIRST = 0, 1
KV_HOST_AUTO, KV_HOST_DIRECT, KV_HOST_STAGED = 0, 1, 2
KV_ORDER_NHD, KV_ORDER_HND = 0, 1
KV_FLAG_VALIDATE, KV_FLAG_IDS_ON_DEVICE = 0x1, 0x2
(KV_OPT_KERNEL, KV_OPT_STAGE_BYTES, KV_OPT_STAGES_PER_WARP, KV_OPT_WARPS, KV_OPT_STORE_LAG,
 KV_OPT_MAX_CTAS, KV_OPT_CHUNK_BYTES, KV_OPT_HOST_MAX_CTAS, KV_OPT_STAGING_SLOTS,
 KV_OPT_L2_HINT, KV_OPT_INLINE_TABLES, KV_OPT_DYNAMIC, KV_OPT_TENSOR_MAPS, KV_OPT_PDL,
 KV_OPT_RESERVE_STAGING, KV_OPT_LEAD_CHUNK) = range(16)
KV_OP_PACK, KV_OP_UNPACK, KV_OP_COW_APPEND = 0, 1, 3
KV_KERNEL_AUTO, KV_KERNEL_BULK, KV_KERNEL_VEC, KV_KERNEL_ELEM, KV_KERNEL_SHOT = 0, 1, 2, 3, 4
(KV_STAT_LAUNCHES, KV_STAT_MEMCPYS, KV_STAT_LAST_ITEMS, KV_STAT_LAST_PAYLOAD, KV_STAT_LAST_KERNEL,
 KV_STAT_LAST_HOST_MODE, KV_STAT_LAST_GRID, KV_STAT_LAST_SEGMENT, KV_STAT_LAST_TENSOR_MAPS, KV_STAT_LAST_PLAIN) = range(10)


class kv_pool_desc(ctypes.Structure):
    _fields_ = [
        ("base", ctypes.POINTER(ctypes.c_void_p)),
        ("layer_count", ctypes.c_uint32),
        ("kv_count", ctypes.c_uint32),
        ("num_pages", ctypes.c_uint32),
        ("page_size", ctypes.c_uint32),
        ("num_heads", ctypes.c_uint32),
        ("head_dim", ctypes.c_uint32),
        ("elem_bytes", ctypes.c_uint32),
        ("order", ctypes.c_uint32),
        ("page_stride_bytes", ctypes.c_uint64),
    ]


class kv_op(ctypes.Structure):
    _fields_ = [
        ("kind", ctypes.c_uint32),
        ("n_pages", ctypes.c_uint32),
        ("page_ids", ctypes.c_void_p),
        ("buf", ctypes.c_void_p),
        ("buf_bytes", ctypes.c_uint64),
        ("n_tokens", ctypes.c_uint64),
        ("n_old", ctypes.c_uint32),
        ("n_app", ctypes.c_uint32),
    ]


_vp, _u32, _u64, _i32, _i64, _int, _sz = (ctypes.c_void_p, ctypes.c_uint32, ctypes.c_uint64,
                                          ctypes.c_int32, ctypes.c_int64, ctypes.c_int,
                                          ctypes.c_size_t)
_pdesc = ctypes.POINTER(kv_pool_desc)


def _sig(name, restype, *argtypes):
    fn = getattr(_lib, name)
    fn.restype = restype
    fn.argtypes = list(argtypes)
    return fn


_kv_version = _sig("kv_version", _u32)
_kv_strerror = _sig("kv_strerror", ctypes.c_char_p, _int)
_kv_ctx_create = _sig("kv_ctx_create", _int, ctypes.POINTER(_vp), _int, _sz)
_kv_ctx_destroy = _sig("kv_ctx_destroy", _int, _vp)
_kv_ctx_set_option = _sig("kv_ctx_set_option", _int, _vp, _int, _i64)
_kv_ctx_get_stat = _sig("kv_ctx_get_stat", _int, _vp, _int, ctypes.POINTER(_u64))
_kv_last_cuda_error = _sig("kv_last_cuda_error", _int, _vp)
_kv_device_status = _sig("kv_device_status", _int, _vp, ctypes.POINTER(_u32))
_kv_peer_enable = _sig("kv_peer_enable", _int, _vp, _int)
_kv_signal = _sig("kv_signal", _int, _vp, _vp, _u64, _vp)
_kv_chain_hash = _sig("kv_chain_hash", _int, _vp, _vp, _vp, _u32, _u32, _vp, _vp, _sz, _vp, _vp)
_kv_host_alloc = _sig("kv_host_alloc", _int, ctypes.POINTER(_vp), _sz)
_kv_host_free = _sig("kv_host_free", _int, _vp)
_kv_host_register = _sig("kv_host_register", _int, _vp, _sz)
_kv_host_unregister = _sig("kv_host_unregister", _int, _vp)
_kv_pack = _sig("kv_pack", _int, _vp, _pdesc, _u32, _vp, _u32, _int, _vp, _sz, _u32, _vp)
_kv_pack_static = _sig("kv_pack_static", _int, _int, _pdesc, _u32, _vp, _u32, _vp, _sz, _vp, ctypes.POINTER(_int))
_kv_unpack = _sig("kv_unpack", _int, _vp, _vp, _sz, _vp, _u32, _pdesc, _u32, _u32, _u32, _u64,
                  _int, _u32, _vp)
_kv_pack_batched = _sig("kv_pack_batched", _int, _vp, _pdesc, _u32, _vp, _vp, _u32, _int, _vp,
                        _vp, _u32, _vp)
_kv_unpack_batched = _sig("kv_unpack_batched", _int, _vp, _vp, _vp, _vp, _vp, _vp, _u32, _pdesc,
                          _u32, _u32, _u32, _int, _u32, _vp)
_kv_offload = _sig("kv_offload", _int, _vp, _pdesc, _u32, _vp, _u32, _int, _vp, _sz, _int, _u32,
                   _vp)
_kv_reload = _sig("kv_reload", _int, _vp, _vp, _sz, _vp, _u32, _pdesc, _u32, _u32, _u32, _u64,
                  _int, _int, _u32, _vp)
_kv_offload_batched = _sig("kv_offload_batched", _int, _vp, _pdesc, _u32, _vp, _vp, _u32, _int,
                           _vp, _vp, _int, _u32, _vp)
_kv_reload_batched = _sig("kv_reload_batched", _int, _vp, _vp, _vp, _vp, _vp, _vp, _u32, _pdesc,
                          _u32, _u32, _u32, _int, _int, _u32, _vp)
_kv_reload_layerwise = _sig("kv_reload_layerwise", _int, _vp, _vp, _sz, _vp, _u32, _pdesc, _u32, _u32, _u32, _u64,
                            _vp, _u64, _int, _u32, _vp)
_kv_reload_layerwise_batched = _sig("kv_reload_layerwise_batched", _int, _vp, _vp, _vp, _vp, _vp, _vp, _u32, _pdesc,
                                    _u32, _u32, _u32, _vp, _u64, _int, _u32, _vp)
_kv_submit = _sig("kv_submit", _int, _vp, _pdesc, _u32, ctypes.POINTER(kv_op), _u32, _int, _u32, _vp)
_kv_repage = _sig("kv_repage", _int, _vp, _pdesc, _vp, _u32, _pdesc, _vp, _u32, _u32, _u64, _u32, _vp)
_kv_repage_batched = _sig("kv_repage_batched", _int, _vp, _pdesc, _vp, _vp, _pdesc, _vp, _vp, _vp,
                          _u32, _u32, _u32, _vp)
_kv_cow_append = _sig("kv_cow_append", _int, _vp, _pdesc, _u32, _i32, _i32, _u32, _vp, _u32, _u32, _vp)
_kv_cow_append_batched = _sig("kv_cow_append_batched", _int, _vp, _pdesc, _u32, _vp, _vp, _vp, _vp,
                              _vp, _u32, _u32, _vp)


class KvError(RuntimeError):
    def __init__(self, status: int, cuda_error: int = 0):
        self.status = status
        self.cuda_error = cuda_error
        msg = kv_strerror(status)
        if cuda_error:
            msg += f" [cudaError {cuda_error}]"
        super().__init__(f"kvtier: {msg} ({status})")


def kv_version() -> int:
    return int(_kv_version())


def kv_strerror(status: int) -> str:
    return _kv_strerror(int(status)).decode()


# ---- marshalling helpers -----------------------------------------------------------------------
def _ptr(x) -> Optional[int]:
    """Address of a torch tensor / numpy array / int / None."""
    if x is None:
        return None
    if type(x) is int:
        return x
    dp = getattr(x, "data_ptr", None)
    if dp is not None:
        return dp()
    if isinstance(x, np.ndarray):
        return x.__array_interface__["data"][0]
    if isinstance(x, int):
        return int(x)
    if isinstance(x, ctypes.c_void_p):
        return x.value
    raise TypeError(f"cannot take the address of {type(x)}")


def _nbytes(x) -> int:
    if hasattr(x, "element_size"):
        return x.numel() * x.element_size()
    if isinstance(x, np.ndarray):
        return int(x.nbytes)
    raise TypeError(f"cannot size {type(x)}; pass nbytes explicitly")


_torch = None
_raw_stream = None  # torch._C._cuda_getCurrentRawStream: the current stream's handle without building a Stream object


def _stream(s, device: int = -1) -> Optional[int]:
    """cudaStream_t of `s` (torch stream / int / None = torch's current stream ON THE CTX'S DEVICE, else the default)."""
    global _torch, _raw_stream
    if s is None:
        if _torch is None:
            try:
                import torch
            except ImportError:
                return None
            _torch = torch
            _raw_stream = getattr(torch._C, "_cuda_getCurrentRawStream", None)
        if _torch.cuda.is_initialized():
            if _raw_stream is not None:
                return _raw_stream(device if device >= 0 else _torch.cuda.current_device()) or None
            return int(_torch.cuda.current_stream(device if device >= 0 else None).cuda_stream) or None
        return None
    if isinstance(s, int):
        return s or None
    return int(s.cuda_stream) or None


_I32 = np.dtype(np.int32)


def _host_i32(a):
    if type(a) is np.ndarray and a.dtype == _I32 and a.flags.c_contiguous:
        return a  # the common case: no copy, no new array object
    return np.ascontiguousarray(np.asarray(a, dtype=np.int32))


def _ids_arg(ids, flags):
    """(pointer, keepalive, count) for a page-id list: host int32 array, or a device tensor when
    KV_FLAG_IDS_ON_DEVICE is set."""
    if flags & KV_FLAG_IDS_ON_DEVICE:
        return _ptr(ids), ids, int(ids.numel())
    a = _host_i32(ids)
    n = a.size
    return (a.__array_interface__["data"][0] if n else None), a, n


class PoolDesc:
    """Owns a kv_pool_desc and its host array of slab base pointers.

    ``slabs`` is a sequence of layer_count*kv_count device pointers (torch tensors or ints) in
    [layer][kv] order (outer dim layers, slice dim K/V); ``order`` is the in-page
    order of the pool, KV_ORDER_NHD [token][head][dim] or KV_ORDER_HND [head][token][dim]."""

    def __init__(self, slabs: Sequence, layer_count: int, kv_count: int, num_pages: int,
                 page_size: int, num_heads: int, head_dim: int, elem_bytes: int,
                 page_stride_bytes: Optional[int] = None, order: int = KV_ORDER_NHD):
        assert len(slabs) == layer_count * kv_count
        self._keep = list(slabs)
        self._base = (ctypes.c_void_p * len(slabs))(*[_ptr(s) for s in slabs])
        row = page_size * num_heads * head_dim * elem_bytes
        self.desc = kv_pool_desc(
            ctypes.cast(self._base, ctypes.POINTER(ctypes.c_void_p)), layer_count, kv_count,
            num_pages, page_size, num_heads, head_dim, elem_bytes, int(order),
            row if page_stride_bytes is None else int(page_stride_bytes))
        self.row_bytes = row
        self.ref = ctypes.byref(self.desc)  # built once: every transfer call passes it

    def page_bytes(self, layer_count: Optional[int] = None) -> int:
        L = self.desc.layer_count if layer_count is None else layer_count
        return L * self.desc.kv_count * self.row_bytes


class Ctx:
    """kv_ctx handle.  ``device=-1`` makes a planning-only context (no CUDA)."""

    def __init__(self, device: int = 0, staging_bytes: int = 0):
        h = ctypes.c_void_p()
        rc = _kv_ctx_create(ctypes.byref(h), int(device), int(staging_bytes))
        if rc:
            raise KvError(rc)
        self.h = h
        self.device = int(device)

    def close(self):
        if getattr(self, "h", None) and _kv_ctx_destroy is not None:
            _kv_ctx_destroy(self.h)
            self.h = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def set_option(self, option: int, value: int):
        rc = _kv_ctx_set_option(self.h, option, value)
        if rc:
            raise KvError(rc)

    def stat(self, stat: int) -> int:
        out = ctypes.c_uint64()
        rc = _kv_ctx_get_stat(self.h, stat, ctypes.byref(out))
        if rc:
            raise KvError(rc)
        return int(out.value)

    def last_cuda_error(self) -> int:
        return int(_kv_last_cuda_error(self.h))

    def device_status(self) -> int:
        out = ctypes.c_uint32()
        rc = _kv_device_status(self.h, ctypes.byref(out))
        if rc:
            raise KvError(rc, self.last_cuda_error())
        return int(out.value)


def _chk(ctx: Ctx, rc: int):
    if rc:
        raise KvError(rc, ctx.last_cuda_error() if rc == KV_ERR_CUDA else 0)


def kv_ctx_create(device: int = 0, staging_bytes: int = 0) -> Ctx:
    return Ctx(device, staging_bytes)


def kv_ctx_destroy(ctx: Ctx):
    ctx.close()


def kv_peer_enable(ctx: Ctx, peer_device: int):
    """Map `peer_device`'s memory into the ctx's device (NVLink P2P); pools/buffers may then live there."""
    _chk(ctx, _kv_peer_enable(ctx.h, int(peer_device)))


def kv_signal(ctx: Ctx, flag, value: int, stream=None):
    """Release-ordered system-scope store of `value` to the 8-byte word `flag` (tensor or address), after
    every transfer already enqueued on the stream."""
    _chk(ctx, _kv_signal(ctx.h, _ptr(flag), int(value), _stream(stream, ctx.device)))


KV_CHAIN_ROOT = 0xCBF29CE484222325


def kv_chain_hash(ctx: Ctx, ident, tok_offsets, page_size: int, out, roots=None, out_capacity=None,
                  stream=None) -> np.ndarray:
    """Chained page ids of all sessions into the device tensor `out`; returns the page
    offsets (int64[S+1]).  `ident` / `out` are device tensors (or addresses), offsets / roots host arrays."""
    off = np.ascontiguousarray(np.asarray(tok_offsets, dtype=np.int64))
    S = max(int(off.size) - 1, 0)
    poff = np.zeros(S + 1, dtype=np.int64)
    r = None if roots is None else _u64_array(roots)
    cap = (int(out.numel()) if hasattr(out, "numel") else 0) if out_capacity is None else int(out_capacity)
    rc = _kv_chain_hash(ctx.h, _ptr(ident), int(off.ctypes.data) if off.size else None, S, int(page_size),
                        None if r is None else int(r.ctypes.data), _ptr(out), cap, int(poff.ctypes.data),
                        _stream(stream, ctx.device))
    _chk(ctx, rc)
    return poff


def kv_host_alloc(nbytes: int) -> int:
    p = ctypes.c_void_p()
    rc = _kv_host_alloc(ctypes.byref(p), int(nbytes))
    if rc:
        raise KvError(rc)
    return int(p.value)


def kv_host_free(p: int):
    rc = _kv_host_free(p)
    if rc:
        raise KvError(rc)


def kv_host_register(p: int, nbytes: int):
    rc = _kv_host_register(p, nbytes)
    if rc:
        raise KvError(rc)


def kv_host_unregister(p: int):
    rc = _kv_host_unregister(p)
    if rc:
        raise KvError(rc)


def host_view(p: int, nbytes: int) -> np.ndarray:
    """numpy uint8 view of pinned memory returned by kv_host_alloc (no copy)."""
    return np.ctypeslib.as_array((ctypes.c_uint8 * nbytes).from_address(p))


def _ptr_array(xs):
    return (ctypes.c_void_p * max(len(xs), 1))(*[_ptr(x) for x in xs])


def _u64_array(xs):
    return np.ascontiguousarray(np.asarray(xs, dtype=np.uint64))


# ---- transfers -------------------------------------------------------------------------------
def kv_pack(ctx: Ctx, pools: PoolDesc, layer_count: int, page_ids, dst, dst_bytes=None,
            layout=KV_LAYOUT_PAGE_FIRST, flags=0, stream=None):
    p, keep, n = _ids_arg(page_ids, flags)
    nb = _nbytes(dst) if dst_bytes is None else int(dst_bytes)
    _chk(ctx, _kv_pack(ctx.h, pools.ref, layer_count, p, n, layout, _ptr(dst), nb, flags,
                       _stream(stream, ctx.device)))


def kv_pack_static(pools: PoolDesc, layer_count: int, page_ids, dst, dst_bytes=None, device: int = 0, stream=None):
    """kv_pack for callers that must not allocate: no Ctx, and the library calls no cudaMalloc / cudaFree on this path.

    Meant for code that runs where an allocation is not an option -- an engine whose KV pools already own the GPU's
    memory, a latency-critical step that cannot afford the device-wide sync of cudaMalloc, a process bound to a fixed
    memory budget.  The lookup tables live in a fixed array inside the library (KV_STATIC_TABLE_BYTES per GPU), so a
    call takes at most KV_STATIC_MAX_PAGES page ids and KV_STATIC_MAX_SLABS layer x K/V slabs (KvError with
    KV_ERR_STATIC_LIMIT beyond that), NHD pools, 16-byte aligned rows, host page ids, page-first layout.  Every call on a
    device shares that array: issue them on one stream (or order them with events); overlapping calls race.  The first
    call on a device looks the array up -- make it before capturing the stream into a CUDA graph.  include/kvtier.h has
    the full contract."""
    a = _host_i32(page_ids)
    n = a.size
    nb = _nbytes(dst) if dst_bytes is None else int(dst_bytes)
    err = _int(0)
    rc = _kv_pack_static(int(device), pools.ref, layer_count, a.__array_interface__["data"][0] if n else None, n,
                         _ptr(dst), nb, _stream(stream, int(device)), ctypes.byref(err))
    if rc:
        raise KvError(rc, int(err.value) if rc == KV_ERR_CUDA else 0)


def kv_unpack(ctx: Ctx, src, dst_page_ids, pools: PoolDesc, layer_count: int, src_page_size: int,
              dst_page_size: int, n_tokens: int, src_bytes=None, layout=KV_LAYOUT_PAGE_FIRST,
              flags=0, stream=None):
    p, keep, n = _ids_arg(dst_page_ids, flags)
    nb = _nbytes(src) if src_bytes is None else int(src_bytes)
    _chk(ctx, _kv_unpack(ctx.h, _ptr(src), nb, p, n, pools.ref, layer_count, src_page_size,
                         dst_page_size, int(n_tokens), layout, flags, _stream(stream, ctx.device)))


def _csr(req_offsets):
    off = np.ascontiguousarray(np.asarray(req_offsets, dtype=np.int64))
    return off, int(off.size - 1)


def kv_pack_batched(ctx: Ctx, pools: PoolDesc, layer_count: int, page_ids, req_offsets, dsts,
                    dst_bytes=None, layout=KV_LAYOUT_PAGE_FIRST, flags=0, stream=None):
    p, keep, _ = _ids_arg(page_ids, flags)
    off, R = _csr(req_offsets)
    d = _ptr_array(dsts)
    nb = None if dst_bytes is None else _u64_array(dst_bytes)
    _chk(ctx, _kv_pack_batched(ctx.h, pools.ref, layer_count, p, off.ctypes.data, R, layout, d,
                               None if nb is None else nb.ctypes.data, flags, _stream(stream, ctx.device)))


def kv_unpack_batched(ctx: Ctx, srcs, dst_page_ids, req_offsets, n_tokens, pools: PoolDesc,
                      layer_count: int, src_page_size: int, dst_page_size: int, src_bytes=None,
                      layout=KV_LAYOUT_PAGE_FIRST, flags=0, stream=None):
    p, keep, _ = _ids_arg(dst_page_ids, flags)
    off, R = _csr(req_offsets)
    s = _ptr_array(srcs)
    nt = _u64_array(n_tokens)
    nb = None if src_bytes is None else _u64_array(src_bytes)
    _chk(ctx, _kv_unpack_batched(ctx.h, s, None if nb is None else nb.ctypes.data, p,
                                 off.ctypes.data, nt.ctypes.data, R, pools.ref, layer_count,
                                 src_page_size, dst_page_size, layout, flags, _stream(stream, ctx.device)))


def kv_offload(ctx: Ctx, pools: PoolDesc, layer_count: int, page_ids, host_dst, host_bytes,
               mode=KV_HOST_AUTO, layout=KV_LAYOUT_PAGE_FIRST, flags=0, stream=None):
    p, keep, n = _ids_arg(page_ids, flags)
    _chk(ctx, _kv_offload(ctx.h, pools.ref, layer_count, p, n, layout, _ptr(host_dst),
                          int(host_bytes), mode, flags, _stream(stream, ctx.device)))


def kv_reload(ctx: Ctx, host_src, host_bytes, dst_page_ids, pools: PoolDesc, layer_count: int,
              src_page_size: int, dst_page_size: int, n_tokens: int, mode=KV_HOST_AUTO,
              layout=KV_LAYOUT_PAGE_FIRST, flags=0, stream=None):
    p, keep, n = _ids_arg(dst_page_ids, flags)
    _chk(ctx, _kv_reload(ctx.h, _ptr(host_src), int(host_bytes), p, n, pools.ref, layer_count,
                         src_page_size, dst_page_size, int(n_tokens), layout, mode, flags,
                         _stream(stream, ctx.device)))


def kv_offload_batched(ctx: Ctx, pools: PoolDesc, layer_count: int, page_ids, req_offsets,
                       host_dsts, host_bytes=None, mode=KV_HOST_AUTO,
                       layout=KV_LAYOUT_PAGE_FIRST, flags=0, stream=None):
    p, keep, _ = _ids_arg(page_ids, flags)
    off, R = _csr(req_offsets)
    d = _ptr_array(host_dsts)
    nb = None if host_bytes is None else _u64_array(host_bytes)
    _chk(ctx, _kv_offload_batched(ctx.h, pools.ref, layer_count, p, off.ctypes.data, R, layout, d,
                                  None if nb is None else nb.ctypes.data, mode, flags,
                                  _stream(stream, ctx.device)))


def kv_reload_batched(ctx: Ctx, host_srcs, dst_page_ids, req_offsets, n_tokens, pools: PoolDesc,
                      layer_count: int, src_page_size: int, dst_page_size: int, host_bytes=None,
                      mode=KV_HOST_AUTO, layout=KV_LAYOUT_PAGE_FIRST, flags=0, stream=None):
    p, keep, _ = _ids_arg(dst_page_ids, flags)
    off, R = _csr(req_offsets)
    s = _ptr_array(host_srcs)
    nt = _u64_array(n_tokens)
    nb = None if host_bytes is None else _u64_array(host_bytes)
    _chk(ctx, _kv_reload_batched(ctx.h, s, None if nb is None else nb.ctypes.data, p,
                                 off.ctypes.data, nt.ctypes.data, R, pools.ref, layer_count,
                                 src_page_size, dst_page_size, layout, mode, flags,
                                 _stream(stream, ctx.device)))


def kv_reload_layerwise(ctx: Ctx, host_src, host_bytes, dst_page_ids, pools: PoolDesc, layer_count: int,
                        src_page_size: int, dst_page_size: int, n_tokens: int, layer_flags, flag_value: int,
                        mode=KV_HOST_AUTO, flags=0, stream=None):
    """Layer-first host buffer -> pool, layer_flags[l] = flag_value stored as each layer lands."""
    p, keep, n = _ids_arg(dst_page_ids, flags)
    _chk(ctx, _kv_reload_layerwise(ctx.h, _ptr(host_src), int(host_bytes), p, n, pools.ref, layer_count,
                                   src_page_size, dst_page_size, int(n_tokens), _ptr(layer_flags),
                                   int(flag_value), mode, flags, _stream(stream, ctx.device)))


def kv_reload_layerwise_batched(ctx: Ctx, host_srcs, dst_page_ids, req_offsets, n_tokens, pools: PoolDesc,
                                layer_count: int, src_page_size: int, dst_page_size: int, layer_flags,
                                flag_value: int, host_bytes=None, mode=KV_HOST_AUTO, flags=0, stream=None):
    p, keep, _ = _ids_arg(dst_page_ids, flags)
    off, R = _csr(req_offsets)
    s = _ptr_array(host_srcs)
    nt = _u64_array(n_tokens)
    nb = None if host_bytes is None else _u64_array(host_bytes)
    _chk(ctx, _kv_reload_layerwise_batched(ctx.h, s, None if nb is None else nb.ctypes.data, p,
                                           off.ctypes.data, nt.ctypes.data, R, pools.ref, layer_count,
                                           src_page_size, dst_page_size, _ptr(layer_flags), int(flag_value),
                                           mode, flags, _stream(stream, ctx.device)))


def op_pack(page_ids, dst, dst_bytes=None):
    """One KV_OP_PACK of kv_submit: gather `page_ids` into the buffer `dst`."""
    return (KV_OP_PACK, page_ids, dst, dst_bytes, 0, 0, 0)


def op_unpack(src, dst_page_ids, n_tokens, src_bytes=None):
    """One KV_OP_UNPACK of kv_submit: scatter the buffer `src` (pool page size) into `dst_page_ids`."""
    return (KV_OP_UNPACK, dst_page_ids, src, src_bytes, int(n_tokens), 0, 0)


def op_cow_append(old_id, new_id, n_old, app, n_app):
    """One KV_OP_COW_APPEND of kv_submit (kv_cow_append's arguments)."""
    return (KV_OP_COW_APPEND, np.array([old_id, new_id], dtype=np.int32), app, 0, 0, int(n_old), int(n_app))


def kv_submit(ctx: Ctx, pools: PoolDesc, layer_count: int, ops, layout=KV_LAYOUT_PAGE_FIRST, flags=0, stream=None):
    """Several independent transfers on one pool in ONE launch; `ops` is a sequence built with op_pack /
    op_unpack / op_cow_append (marshalled into the C array of kv_op)."""
    n = len(ops)
    arr = (kv_op * max(n, 1))()
    keep = []
    for i, (kind, ids, buf, nbytes, n_tokens, n_old, n_app) in enumerate(ops):
        a = _host_i32(ids)
        keep.append(a)
        o = arr[i]
        o.kind = kind
        o.n_pages = 0 if kind == KV_OP_COW_APPEND else a.size
        o.page_ids = a.__array_interface__["data"][0] if a.size else None
        o.buf = _ptr(buf)
        o.buf_bytes = 0 if kind == KV_OP_COW_APPEND else (_nbytes(buf) if nbytes is None else int(nbytes))
        o.n_tokens = n_tokens
        o.n_old, o.n_app = n_old, n_app
    _chk(ctx, _kv_submit(ctx.h, pools.ref, layer_count, arr, n, layout, flags, _stream(stream, ctx.device)))


def kv_repage(ctx: Ctx, src_pools: PoolDesc, src_page_ids, dst_pools: PoolDesc, dst_page_ids,
              layer_count: int, n_tokens: int, flags=0, stream=None):
    sp, skeep, ns = _ids_arg(src_page_ids, flags)
    dp, dkeep, nd = _ids_arg(dst_page_ids, flags)
    _chk(ctx, _kv_repage(ctx.h, src_pools.ref, sp, ns, dst_pools.ref, dp, nd, layer_count,
                         int(n_tokens), flags, _stream(stream, ctx.device)))


def kv_repage_batched(ctx: Ctx, src_pools: PoolDesc, src_page_ids, src_offsets, dst_pools: PoolDesc,
                      dst_page_ids, dst_offsets, n_tokens, layer_count: int, flags=0, stream=None):
    sp, skeep, _ = _ids_arg(src_page_ids, flags)
    dp, dkeep, _ = _ids_arg(dst_page_ids, flags)
    soff, R = _csr(src_offsets)
    doff, R2 = _csr(dst_offsets)
    assert R == R2
    nt = _u64_array(n_tokens)
    _chk(ctx, _kv_repage_batched(ctx.h, src_pools.ref, sp, soff.ctypes.data, dst_pools.ref, dp,
                                 doff.ctypes.data, nt.ctypes.data, R, layer_count, flags,
                                 _stream(stream, ctx.device)))


def kv_cow_append(ctx: Ctx, pools: PoolDesc, layer_count: int, old_id: int, new_id: int, n_old: int,
                  app, n_app: int, flags=0, stream=None):
    _chk(ctx, _kv_cow_append(ctx.h, pools.ref, layer_count, int(old_id), int(new_id), int(n_old),
                             _ptr(app), int(n_app), flags, _stream(stream, ctx.device)))


def kv_cow_append_batched(ctx: Ctx, pools: PoolDesc, layer_count: int, old_ids, new_ids, n_old,
                          n_app, apps, flags=0, stream=None):
    no = np.ascontiguousarray(np.asarray(n_old, dtype=np.uint32))
    na = np.ascontiguousarray(np.asarray(n_app, dtype=np.uint32))
    S = int(no.size)
    if flags & KV_FLAG_IDS_ON_DEVICE:  # device tensors of S int32 ids each
        op, np_ = _ptr(old_ids), _ptr(new_ids)
        assert int(old_ids.numel()) == S and int(new_ids.numel()) == S
    else:
        o, n = _host_i32(old_ids), _host_i32(new_ids)
        assert o.size == S and n.size == S
        op, np_ = (o.ctypes.data if S else None), (n.ctypes.data if S else None)
    assert na.size == S and len(apps) == S
    a = _ptr_array(apps)
    _chk(ctx, _kv_cow_append_batched(ctx.h, pools.ref, layer_count, op, np_, no.ctypes.data if S else None,
                                     na.ctypes.data if S else None, a, S, flags, _stream(stream, ctx.device)))
