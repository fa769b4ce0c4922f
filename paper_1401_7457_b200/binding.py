"""ctypes binding of include/cx_bwt.h: same names, argument marshalling only.

PyTorch supplies device memory and streams; every step of the path runs in libcxbwt.so.  There is no
fallback: if the library is missing and cannot be built, or a call fails, this raises.
"""
from __future__ import annotations

import ctypes
import os

import torch

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))

CX_OK, CX_ERR_ARG, CX_ERR_BAD_BASE, CX_ERR_WORKSPACE, CX_ERR_BUCKET_TOO_LARGE, CX_ERR_CUDA, CX_ERR_NOMEM = 0, -1, -2, -3, -4, -5, -6
KERNEL_CLASSES = ["pack", "prep", "hist", "list", "sort_hist", "sort_scan", "sort_pass", "finish", "refine_scan", "refine_key",
                  "refine_write", "refine_sort", "finish_block"]


class CxError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"cx error {code}: {text}")
        self.code = code


class cx_bwt_opts_t(ctypes.Structure):
    _fields_ = [("prefix_len", ctypes.c_uint32), ("key_bases", ctypes.c_uint32), ("max_batch_suffixes", ctypes.c_uint64),
                ("max_read_len", ctypes.c_uint32), ("out_is_host_pinned", ctypes.c_int32), ("small_group_max", ctypes.c_uint32),
                ("profile", ctypes.c_uint32), ("finish_slots", ctypes.c_uint32), ("out_bits", ctypes.c_uint32), ("shard_index", ctypes.c_uint32), ("shard_count", ctypes.c_uint32)]


class cx_bwt_stats_t(ctypes.Structure):
    _fields_ = [("n_suffixes", ctypes.c_uint64), ("max_batch", ctypes.c_uint64), ("largest_bucket", ctypes.c_uint64),
                ("refine_elements", ctypes.c_uint64), ("small_group_elems", ctypes.c_uint64), ("kernel_launches", ctypes.c_uint64), ("compare_ops", ctypes.c_uint64),
                ("n_batches", ctypes.c_uint32), ("id_bytes", ctypes.c_uint32), ("sort_passes", ctypes.c_uint32),
                ("refine_rounds", ctypes.c_uint32), ("max_read_len", ctypes.c_uint32), ("uniform_len", ctypes.c_uint32), ("refined_partitions", ctypes.c_uint32),
                ("shard_offset", ctypes.c_uint64), ("shard_suffixes", ctypes.c_uint64), ("finish_rounds", ctypes.c_uint64)]

    def as_dict(self) -> dict:
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


_lib = None


def lib() -> ctypes.CDLL:
    """Load (building first if stale) libcxbwt.so.  Fails loudly; never substitutes another path."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        vp, u64, u32, i32 = ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint32, ctypes.c_int
        L.cx_bwt_workspace_bytes.argtypes = [u64, u64, ctypes.POINTER(cx_bwt_opts_t), ctypes.POINTER(u64)]
        L.cx_bwt_plan.argtypes = [ctypes.POINTER(vp), u64, u64, ctypes.POINTER(cx_bwt_opts_t), vp, u64]
        L.cx_pack_reads.argtypes = [vp, u64, vp, vp, vp]
        L.cx_bwt_build.argtypes = [vp, vp, vp, u64, vp, vp]
        L.cx_bwt_free.argtypes = [vp]
        L.cx_bwt_get_stats.argtypes = [vp, ctypes.POINTER(cx_bwt_stats_t)]
        L.cx_bwt_get_histogram.argtypes = [vp, vp, u64, ctypes.POINTER(u64)]
        L.cx_bwt_kernel_time.argtypes = [vp, i32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(u64), ctypes.POINTER(u64)]
        L.cx_sort_pairs_workspace_bytes.argtypes = [u64, ctypes.POINTER(u64)]
        L.cx_sort_pairs.argtypes = [vp, vp, vp, vp, u64, u32, u32, u32, vp, u64, ctypes.POINTER(i32), vp]
        L.cx_fasta_workspace_bytes.argtypes = [u64, ctypes.POINTER(u64)]
        L.cx_fasta_parse.argtypes = [vp, u64, vp, vp, u64, vp, vp, u64, vp]
        L.cx_sort_pairs_static.argtypes = [vp, vp, vp, vp, u64, u32, u32, u32, ctypes.POINTER(i32), vp]
        L.cx_sort_pairs_static.restype = i32
        L.cx_strerror_static.argtypes = []
        L.cx_strerror_static.restype = ctypes.c_char_p
        L.cx_strerror.argtypes = [i32]
        L.cx_strerror.restype = ctypes.c_char_p
        for name in ("cx_bwt_workspace_bytes", "cx_bwt_plan", "cx_pack_reads", "cx_bwt_build", "cx_bwt_free", "cx_bwt_get_stats",
                     "cx_bwt_get_histogram", "cx_bwt_kernel_time", "cx_sort_pairs_workspace_bytes", "cx_sort_pairs",
                     "cx_fasta_workspace_bytes", "cx_fasta_parse"):
            getattr(L, name).restype = i32
        _lib = L
    return _lib


def cx_strerror(code: int) -> str:
    return lib().cx_strerror(code).decode()


def _check(rc: int) -> None:
    if rc != CX_OK:
        raise CxError(rc, cx_strerror(rc))


def _stream_ptr(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream


def _opts(**kw) -> cx_bwt_opts_t:
    o = cx_bwt_opts_t()
    for k, v in kw.items():
        if v is not None:
            setattr(o, k, int(v))
    return o


def cx_bwt_workspace_bytes(n_reads: int, total_bases: int, **opts) -> int:
    out = ctypes.c_uint64(0)
    o = _opts(**opts)
    _check(lib().cx_bwt_workspace_bytes(n_reads, total_bases, ctypes.byref(o), ctypes.byref(out)))
    return int(out.value)


def cx_pack_reads(ascii_dev: torch.Tensor, packed_out: torch.Tensor | None = None, stream=None, check: bool = True,
                  status: torch.Tensor | None = None) -> torch.Tensor:
    """ASCII bases (uint8, cuda) -> packed words (int64 tensor holding uint64 bit patterns).

    check=True reads the status word back (one synchronisation) and raises CX_ERR_BAD_BASE; with check=False the
    call is fully asynchronous and the caller inspects `status` (count of warps that saw a byte outside ACGT)."""
    assert ascii_dev.is_cuda and ascii_dev.dtype == torch.uint8 and ascii_dev.is_contiguous()
    n = ascii_dev.numel()
    if packed_out is None:
        packed_out = torch.empty(max(1, (n + 31) // 32), dtype=torch.int64, device=ascii_dev.device)
    if status is None:
        status = _pack_status(ascii_dev.device)
    with torch.cuda.device(ascii_dev.device):
        _check(lib().cx_pack_reads(ascii_dev.data_ptr(), n, packed_out.data_ptr(), status.data_ptr(), _stream_ptr(stream)))
    if check and int(status.item()) != 0:
        raise CxError(CX_ERR_BAD_BASE, cx_strerror(CX_ERR_BAD_BASE))
    return packed_out


_copy_streams: dict = {}


def pack_reads_from_host(ascii_host: torch.Tensor, ascii_dev: torch.Tensor, packed_out: torch.Tensor, stream=None,
                         chunk_bytes: int = 64 << 20) -> torch.Tensor:
    """Ingest from pinned HOST memory: the ASCII bases are copied to the device in chunks on a side stream while
    cx_pack_reads packs the chunks that have already arrived (copies and calls only: the packing is the kernel's).
    Chunks are multiples of 32 bases, so every chunk starts a packed word."""
    assert ascii_host.dtype == torch.uint8 and ascii_host.is_pinned() and ascii_dev.is_cuda and ascii_dev.numel() >= ascii_host.numel()
    n = ascii_host.numel()
    main = torch.cuda.current_stream() if stream is None else stream
    key = str(ascii_dev.device)
    if key not in _copy_streams:
        _copy_streams[key] = torch.cuda.Stream(device=ascii_dev.device)
    side = _copy_streams[key]
    side.wait_stream(main)                                # the buffers may still be in use by earlier work on `main`
    status = _pack_status(ascii_dev.device)
    chunk = max(32, chunk_bytes // 32 * 32)
    for a in range(0, n, chunk):
        b = min(n, a + chunk)
        with torch.cuda.stream(side):
            ascii_dev[a:b].copy_(ascii_host[a:b], non_blocking=True)
            ev = torch.cuda.Event()
            ev.record(side)
        main.wait_event(ev)
        with torch.cuda.device(ascii_dev.device):
            _check(lib().cx_pack_reads(ascii_dev.data_ptr() + a, b - a, packed_out.data_ptr() + (a // 32) * 8, status.data_ptr(), main.cuda_stream))
    return packed_out


class HostPipeline:
    """Back-to-back builds from pinned HOST memory with the copies of neighbouring builds overlapped (copies and calls
    only): while collection i is built, collection i + 1 is copied in and packed on a second stream and the output of
    collection i - 1 is copied to pinned host memory on a third.  Two sets of device buffers, one plan.

    `run(collections)` takes an iterable of (ascii_host, offsets_host, n_reads) -- pinned uint8 / int64 tensors -- and
    yields one pinned uint8 tensor per collection, in order.  A yielded tensor is overwritten two collections later:
    use it (or copy it) before asking for the result after the next.  This is a THROUGHPUT arrangement: the time from
    a collection's first byte in to its last byte out is longer than with a single build, not shorter."""

    def __init__(self, plan: "Plan", max_reads: int, max_total_bases: int):
        dev = plan.device
        # the pipeline copies whole 8-bit outputs itself; a plan that streams to the host or packs its output is used on its own
        if plan.opts.out_is_host_pinned or plan.opts.out_bits not in (0, 8) or plan.opts.shard_count > 1:
            raise CxError(CX_ERR_ARG, "HostPipeline needs a plan with device output, 8-bit symbols and no sharding")
        self.plan, self.device = plan, dev
        self.s_in, self.s_out = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
        n_out = max_total_bases + max_reads
        self.sets = [dict(ascii=torch.empty(max(1, max_total_bases), dtype=torch.uint8, device=dev),
                          packed=torch.empty((max_total_bases + 31) // 32 + 1, dtype=torch.int64, device=dev),
                          off=torch.empty(max_reads + 1, dtype=torch.int64, device=dev),
                          out=torch.empty(max(1, n_out), dtype=torch.uint8, device=dev),
                          host=torch.empty(max(1, n_out), dtype=torch.uint8).pin_memory(),
                          in_ready=None, built=None, copied=None) for _ in range(2)]

    def _load(self, b: int, item) -> None:
        ascii_host, offsets_host, n_reads = item
        st = self.sets[b]
        assert offsets_host.dtype == torch.int64 and offsets_host.is_pinned() and offsets_host.numel() == n_reads + 1
        if st["built"] is not None:
            self.s_in.wait_event(st["built"])            # the build that read this set is done
        with torch.cuda.stream(self.s_in):
            pack_reads_from_host(ascii_host, st["ascii"], st["packed"], stream=self.s_in)
            st["off"][:n_reads + 1].copy_(offsets_host, non_blocking=True)
        st["in_ready"] = torch.cuda.Event()
        st["in_ready"].record(self.s_in)

    def run(self, collections):
        main = torch.cuda.current_stream(self.device)
        it = iter(collections)
        nxt = next(it, None)
        if nxt is not None:
            self._load(0, nxt)
        i, pending = 0, None
        while nxt is not None:
            cur, st = nxt, self.sets[i & 1]
            nxt = next(it, None)
            main.wait_event(st["in_ready"])
            if nxt is not None:
                self._load((i & 1) ^ 1, nxt)             # the next collection arrives while this one is built
            if st["copied"] is not None:
                main.wait_event(st["copied"])            # this set's previous output has left the device
            n_reads, n_out = cur[2], cur[0].numel() + cur[2]
            self.plan.build(st["packed"], st["off"], n_reads, st["out"], stream=main)
            st["built"] = torch.cuda.Event()
            st["built"].record(main)
            self.s_out.wait_event(st["built"])
            with torch.cuda.stream(self.s_out):
                st["host"][:n_out].copy_(st["out"][:n_out], non_blocking=True)
            st["copied"] = torch.cuda.Event()
            st["copied"].record(self.s_out)
            if pending is not None:
                pending[1].synchronize()
                yield pending[0]
            pending = (st["host"][:n_out], st["copied"])
            i += 1
        if pending is not None:
            pending[1].synchronize()
            yield pending[0]


_status_words: dict = {}


def _pack_status(device) -> torch.Tensor:
    key = str(device)
    if key not in _status_words:
        _status_words[key] = torch.zeros(1, dtype=torch.int32, device=device)
    return _status_words[key]


class Plan:
    """cx_bwt_plan / cx_bwt_build / cx_bwt_free with a torch-owned workspace."""

    def __init__(self, max_reads: int, max_total_bases: int, workspace_bytes: int | None = None, device=None, **opts):
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self.opts = _opts(**opts)
        if workspace_bytes is None:
            workspace_bytes = cx_bwt_workspace_bytes(max_reads, max_total_bases, **opts)
        self.workspace = torch.empty(int(workspace_bytes) + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        self._ws_ptr = (base + 255) // 256 * 256
        self._h = ctypes.c_void_p(None)
        with torch.cuda.device(self.device):
            _check(lib().cx_bwt_plan(ctypes.byref(self._h), max_reads, max_total_bases, ctypes.byref(self.opts), self._ws_ptr,
                                     int(workspace_bytes)))

    def build(self, packed: torch.Tensor, offsets: torch.Tensor, n_reads: int, out: torch.Tensor, stream=None) -> torch.Tensor:
        """cx_bwt_build: out receives N = total_bases + n_reads bytes over b"$ACGT"."""
        assert offsets.dtype == torch.int64 and offsets.is_cuda and offsets.is_contiguous()
        assert out.dtype == torch.uint8 and out.is_contiguous()
        with torch.cuda.device(self.device):
            _check(lib().cx_bwt_build(self._h, packed.data_ptr(), offsets.data_ptr(), n_reads, out.data_ptr(), _stream_ptr(stream)))
        return out

    def stats(self) -> dict:
        s = cx_bwt_stats_t()
        _check(lib().cx_bwt_get_stats(self._h, ctypes.byref(s)))
        return s.as_dict()

    def histogram(self):
        import numpy as np
        n = ctypes.c_uint64(0)
        lib().cx_bwt_get_histogram(self._h, None, 0, ctypes.byref(n))
        h = np.zeros(int(n.value), dtype=np.uint64)
        _check(lib().cx_bwt_get_histogram(self._h, h.ctypes.data, h.shape[0], ctypes.byref(n)))
        return h

    def kernel_times(self) -> dict:
        out = {}
        for i, name in enumerate(KERNEL_CLASSES):
            ms, ln, by = ctypes.c_double(0), ctypes.c_uint64(0), ctypes.c_uint64(0)
            _check(lib().cx_bwt_kernel_time(self._h, i, ctypes.byref(ms), ctypes.byref(ln), ctypes.byref(by)))
            out[name] = {"ms": ms.value, "launches": int(ln.value), "bytes": int(by.value)}
        return out

    def free(self) -> None:
        if self._h:
            lib().cx_bwt_free(self._h)
            self._h = ctypes.c_void_p(None)

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def cx_sort_pairs(keys: torch.Tensor, vals: torch.Tensor, begin_bit: int = 0, end_bit: int = 64, stream=None):
    """Stable LSD radix sort of (uint64 key as int64 bits, 4- or 8-byte value) pairs; returns new tensors."""
    assert keys.is_cuda and keys.dtype == torch.int64 and vals.dtype in (torch.int32, torch.int64)
    n = keys.numel()
    k0, v0 = keys.clone(), vals.clone()
    k1, v1 = torch.empty_like(k0), torch.empty_like(v0)
    wsb = ctypes.c_uint64(0)
    _check(lib().cx_sort_pairs_workspace_bytes(n, ctypes.byref(wsb)))
    ws = torch.empty(int(wsb.value), dtype=torch.uint8, device=keys.device)
    alt = ctypes.c_int(0)
    _check(lib().cx_sort_pairs(k0.data_ptr(), v0.data_ptr(), k1.data_ptr(), v1.data_ptr(), n, vals.element_size(), begin_bit,
                               end_bit, ws.data_ptr(), int(wsb.value), ctypes.byref(alt), _stream_ptr(stream)))
    return (k1, v1) if alt.value else (k0, v0)


CX_SORT_STATIC_MAX_PAIRS = 1 << 20


def cx_sort_pairs_static(keys: torch.Tensor, vals: torch.Tensor, keys_alt: torch.Tensor, vals_alt: torch.Tensor, begin_bit: int = 0,
                         end_bit: int = 64, stream=None):
    """cx_sort_pairs_static: sorts in place over the caller's double buffers (keys/vals are overwritten); the library's static
    device scratch serves as workspace, so nothing is allocated here or in the library.  Returns the pair of tensors that holds
    the result.  n <= CX_SORT_STATIC_MAX_PAIRS, else CxError(CX_ERR_ARG)."""
    assert keys.is_cuda and keys.dtype == torch.int64 and vals.dtype in (torch.int32, torch.int64)
    assert keys_alt.shape == keys.shape and vals_alt.shape == vals.shape and keys_alt.dtype == keys.dtype and vals_alt.dtype == vals.dtype
    alt = ctypes.c_int(0)
    with torch.cuda.device(keys.device):
        rc = lib().cx_sort_pairs_static(keys.data_ptr(), vals.data_ptr(), keys_alt.data_ptr(), vals_alt.data_ptr(), keys.numel(), vals.element_size(),
                                        begin_bit, end_bit, ctypes.byref(alt), _stream_ptr(stream))
    if rc != CX_OK:
        raise CxError(rc, lib().cx_strerror_static().decode())
    return (keys_alt, vals_alt) if alt.value else (keys, vals)


def cx_fasta_parse(text_dev: torch.Tensor, max_reads: int | None = None, stream=None):
    """cx_fasta_parse: FASTA text (uint8, device) -> (bases uint8[total], read_offsets int64[n_reads + 1]), both on the device.
    max_reads bounds the offsets buffer (default: one read per two bytes of text, the most a FASTA text can hold)."""
    assert text_dev.is_cuda and text_dev.dtype == torch.uint8 and text_dev.is_contiguous()
    n = text_dev.numel()
    if max_reads is None:
        max_reads = n // 2 + 1
    wsb = ctypes.c_uint64(0)
    _check(lib().cx_fasta_workspace_bytes(n, ctypes.byref(wsb)))
    ws = torch.empty(int(wsb.value) + 256, dtype=torch.uint8, device=text_dev.device)
    ws_ptr = (ws.data_ptr() + 255) // 256 * 256
    bases = torch.empty(max(n, 1), dtype=torch.uint8, device=text_dev.device)
    offsets = torch.empty(max_reads + 1, dtype=torch.int64, device=text_dev.device)
    counts = torch.empty(3, dtype=torch.int64, device=text_dev.device)
    with torch.cuda.device(text_dev.device):
        _check(lib().cx_fasta_parse(text_dev.data_ptr(), n, bases.data_ptr(), offsets.data_ptr(), max_reads, counts.data_ptr(), ws_ptr,
                                    int(wsb.value), _stream_ptr(stream)))
        n_reads, total, orphans = (int(x) for x in counts.cpu())     # synchronises
    if orphans:
        raise CxError(-1, f"not FASTA: {orphans} sequence bytes before the first '>' header")
    if n_reads > max_reads:
        raise CxError(-1, f"{n_reads} reads in the text, max_reads = {max_reads}")
    return bases[:total], offsets[:n_reads + 1]


def bwt_of_fasta(text_host, device="cuda", **opts):
    """Host FASTA bytes -> host BWT bytes (numpy): H2D copy, cx_fasta_parse, cx_pack_reads, cx_bwt_build, D2H copy."""
    import numpy as np
    t = torch.from_numpy(np.frombuffer(bytes(text_host), dtype=np.uint8).copy()).to(device)
    bases, offsets = cx_fasta_parse(t)
    n_reads, total = offsets.numel() - 1, bases.numel()
    if n_reads <= 0:
        return np.zeros(0, dtype=np.uint8)
    packed = cx_pack_reads(bases) if total else torch.zeros(1, dtype=torch.int64, device=device)
    opts.setdefault("max_read_len", max(int((offsets[1:] - offsets[:-1]).max()), 1))
    plan = Plan(n_reads, total, **opts)
    out = torch.empty(total + n_reads, dtype=torch.uint8, device=device)
    plan.build(packed, offsets, n_reads, out)
    res = out.cpu().numpy()
    plan.free()
    return res


def bwt_of_collection(ascii_host, offsets_host, device="cuda", **opts):
    """The call a user makes: host ASCII reads + offsets -> host BWT bytes (numpy), through pack + build."""
    import numpy as np
    n_reads = int(offsets_host.shape[0] - 1)
    total = int(offsets_host[-1]) if n_reads > 0 else 0
    N = total + n_reads
    if n_reads <= 0:
        return np.zeros(0, dtype=np.uint8)
    a = torch.from_numpy(np.ascontiguousarray(ascii_host)).to(device) if total else torch.zeros(0, dtype=torch.uint8, device=device)
    off = torch.from_numpy(np.ascontiguousarray(offsets_host).astype(np.int64)).to(device)
    packed = cx_pack_reads(a) if total else torch.zeros(1, dtype=torch.int64, device=device)
    plan = Plan(n_reads, total, **opts)
    out = torch.empty(N, dtype=torch.uint8, device=device)
    plan.build(packed, off, n_reads, out)
    res = out.cpu().numpy()
    plan.free()
    return res
