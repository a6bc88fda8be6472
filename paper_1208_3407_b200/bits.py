"""Thin Python binding of the C ABI in include/bits.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of libbits_b200.so; PyTorch supplies device
memory and the current CUDA stream and nothing else.  There is no CPU fallback: if the library
is missing or the call fails, a BitsError is raised.

Function names mirror the C entry points: count, count_per_interval, mc_rounds, place,
sort_u32 (device tensors in, device tensors out) and count_host, count_per_interval_host,
mc_rounds_host (host arrays in, host arrays out, copies inside the call).
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np
import torch

from . import build as _build

PERMUTE_A, PERMUTE_B = 0, 1
B_SORTED, VALIDATE = 1, 2
FN_COUNT, FN_COUNT_PER_INTERVAL, FN_MC_ROUNDS, FN_PLACE, FN_SORT, FN_ENUMERATE = 0, 1, 2, 3, 4, 5

_u32p, _u64p, _vp = C.c_void_p, C.c_void_p, C.c_void_p   # raw addresses (host or device)
_lib = None

_SIGNATURES = {
    "bits_workspace_bytes": (C.c_size_t, [C.c_int, C.c_uint64, C.c_uint64, C.c_uint32, C.c_int, C.c_uint32]),
    "bits_workspace_sorted_offset": (C.c_int, [C.c_int, C.c_uint64, C.c_uint64, C.c_uint32, C.c_int, C.c_int, C.c_void_p]),
    "bits_host_staging_bytes": (C.c_size_t, [C.c_int, C.c_uint64, C.c_uint64, C.c_uint32]),
    "bits_count": (C.c_int, [_u32p, _u32p, C.c_uint64, _u32p, _u32p, C.c_uint64, C.c_uint32, _vp, C.c_size_t,
                             _u64p, _vp]),
    "bits_count_static": (C.c_int, [_u32p, _u32p, C.c_uint64, _u32p, _u32p, C.c_uint64, C.c_uint32, _u64p, _vp]),
    "bits_decide": (C.c_int, [_u32p, _u32p, C.c_uint64, _u32p, _u32p, C.c_uint64, C.c_uint32, _vp, C.c_size_t, _u32p, _vp]),
    "bits_enumerate": (C.c_int, [_u32p, _u32p, C.c_uint64, _u32p, _u32p, C.c_uint64, C.c_uint32, _vp, C.c_size_t, _u32p, _u32p,
                                 C.c_uint64, _u64p, _vp]),
    "bits_count_per_interval": (C.c_int, [_u32p, _u32p, C.c_uint64, _u32p, _u32p, C.c_uint64, C.c_uint32, _vp,
                                          C.c_size_t, _u32p, _u64p, _vp]),
    "bits_mc_rounds": (C.c_int, [_u32p, _u32p, C.c_uint64, _u32p, _u32p, C.c_uint64, _u32p, C.c_uint32, C.c_int,
                                 C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, _vp, C.c_size_t, _u64p, _u64p, _vp]),
    "bits_place": (C.c_int, [_u32p, C.c_uint64, _u32p, C.c_uint32, C.c_uint64, C.c_uint32, C.c_uint32, _vp,
                             C.c_size_t, _u32p, _u32p, _vp]),
    "bits_sort_u32": (C.c_int, [_u32p, _u32p, C.c_uint64, _vp, C.c_size_t, _vp]),
    "bits_count_host": (C.c_int, [_u32p, _u32p, C.c_uint64, _u32p, _u32p, C.c_uint64, C.c_uint32, _vp, C.c_size_t,
                                  _u64p, _vp]),
    "bits_count_per_interval_host": (C.c_int, [_u32p, _u32p, C.c_uint64, _u32p, _u32p, C.c_uint64, C.c_uint32, _vp,
                                               C.c_size_t, _u32p, _u64p, _vp]),
    "bits_mc_rounds_host": (C.c_int, [_u32p, _u32p, C.c_uint64, _u32p, _u32p, C.c_uint64, _u32p, C.c_uint32, C.c_int,
                                      C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, _vp, C.c_size_t, _u64p, _u64p,
                                      _vp]),
    "bits_pvalue": (C.c_double, [C.c_uint64, _u64p, C.c_uint32, C.c_int]),
    "bits_enrichment": (C.c_double, [C.c_uint64, _u64p, C.c_uint32]),
    "bits_screen_workspace_bytes": (C.c_size_t, [C.c_void_p, C.c_uint32, C.c_uint32]),
    "bits_screen": (C.c_int, [_u32p, _u32p, C.c_void_p, C.c_uint32, _u32p, C.c_uint32, C.c_uint64, C.c_uint32, C.c_uint32,
                              C.c_uint32, _vp, C.c_size_t, _u64p, _u64p, _vp]),
    "bits_screen_enrichment": (C.c_int, [_u64p, _u64p, C.c_uint64, C.c_uint32, C.c_void_p]),
    "bits_launch_count": (C.c_uint64, []),
    "bits_profile_read": (C.c_int, [C.c_int, C.c_void_p, C.c_void_p]),
    "bits_set_option": (C.c_int, [C.c_char_p, C.c_int64]),
    "bits_strerror": (C.c_char_p, [C.c_int]),
    "bits_version": (C.c_char_p, []),
}
EXPORTS = tuple(_SIGNATURES)


class BitsError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"bits status {status}: {msg}")
        self.status = status


def lib_path() -> str:
    return _build.LIB


def lib():
    """Load libbits_b200.so (building it with nvcc if it is stale or missing).  Fails loudly."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(L, name)          # AttributeError if a declared symbol is not exported
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _chk(status: int):
    if status != 0:
        raise BitsError(status, lib().bits_strerror(status).decode())


def strerror(status: int) -> str:
    return lib().bits_strerror(status).decode()


def version() -> str:
    return lib().bits_version().decode()


def launch_count() -> int:
    return int(lib().bits_launch_count())


def set_option(name: str, value: int) -> None:
    _chk(lib().bits_set_option(name.encode(), int(value)))


PROFILE_CLASSES = ("place", "histogram", "sort_pass", "index_build", "count", "sorted_query", "mc_permute_a", "other",
                   "plan", "scatter", "bucket_sort", "place_scatter", "bucket_sort_search", "query_scatter", "bucket_search")


def profile_read() -> dict:
    """{class: (milliseconds, launches)} accumulated while set_option("profile", 1) was on."""
    out = {}
    for i, name in enumerate(PROFILE_CLASSES):
        ms, n = C.c_double(0), C.c_uint64(0)
        _chk(lib().bits_profile_read(i, C.addressof(ms), C.addressof(n)))
        out[name] = (ms.value, int(n.value))
    return out


def workspace_bytes(fn: int, n_a: int, n_b: int, n_chrom: int = 0, which: int = 0, flags: int = 0) -> int:
    return int(lib().bits_workspace_bytes(fn, n_a, n_b, n_chrom, which, flags))


def sorted_arrays_in_workspace(ws: torch.Tensor, fn: int, n_a: int, n_b: int, n_chrom: int = 0, which: int = 0):
    """(B_S, B_E) views into a workspace the call `fn` ran with (bits_workspace_sorted_offset)."""
    out = []
    for array in (0, 1):
        off = C.c_size_t(0)
        _chk(lib().bits_workspace_sorted_offset(fn, n_a, n_b, n_chrom, which, array, C.addressof(off)))
        out.append(ws[off.value: off.value + 4 * n_b].view(torch.int32))
    return tuple(out)


def host_staging_bytes(fn: int, n_a: int, n_b: int, n_rounds: int = 0) -> int:
    return int(lib().bits_host_staging_bytes(fn, n_a, n_b, n_rounds))


# --------------------------------------------------------------------------------------------
def _dev_u32(t: torch.Tensor, name: str) -> int:
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.element_size() == 4
            and not t.dtype.is_floating_point and t.dim() == 1):
        raise TypeError(f"{name}: expected a contiguous 1-D 32-bit integer CUDA tensor")
    return t.data_ptr() if t.numel() else 0


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _workspace(nbytes: int, workspace: torch.Tensor | None, device) -> torch.Tensor:
    if workspace is None:
        workspace = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=device)
    if workspace.numel() * workspace.element_size() < nbytes:
        raise BitsError(5, "workspace tensor too small")
    return workspace


def _host_u32(x, name: str) -> np.ndarray:
    if isinstance(x, torch.Tensor):
        if x.is_cuda:
            raise TypeError(f"{name}: expected host memory")
        x = x.numpy()
    a = np.ascontiguousarray(x)
    if a.dtype != np.uint32:
        if a.dtype.itemsize == 4 and a.dtype.kind in "iu":
            a = a.view(np.uint32)
        else:
            a = a.astype(np.uint32)
    return a


def _offsets(chrom_offsets) -> np.ndarray:
    off = np.ascontiguousarray(np.asarray(chrom_offsets), dtype=np.uint32)
    if off.ndim != 1 or off.size < 2:
        raise BitsError(3, "chromosome offset table needs at least two entries")
    return off


def count(a_start, a_end, b_start, b_end, flags: int = 0, workspace=None, total_out=None) -> torch.Tensor:
    """bits_count -> device int64[1] tensor holding the uint64 total (valid after stream sync)."""
    dev = a_start.device
    n_a, n_b = a_start.numel(), b_start.numel()
    ws = _workspace(workspace_bytes(FN_COUNT, n_a, n_b, 0, 0, flags), workspace, dev)
    out = total_out if total_out is not None else torch.empty(1, dtype=torch.int64, device=dev)
    _chk(lib().bits_count(_dev_u32(a_start, "a_start"), _dev_u32(a_end, "a_end"), n_a,
                          _dev_u32(b_start, "b_start"), _dev_u32(b_end, "b_end"), n_b, flags,
                          ws.data_ptr(), ws.numel(), out.data_ptr(), _stream()))
    return out


STATIC_SCRATCH_BYTES = 32 << 20     # BITS_STATIC_SCRATCH_BYTES of include/bits.h


def count_static(a_start, a_end, b_start, b_end, flags: int = 0, total_out=None) -> torch.Tensor:
    """bits_count_static -> device int64[1] tensor holding the uint64 total (valid after stream sync).

    bits_count for callers that cannot allocate a workspace (a stage inside an application that owns all device
    memory, a path on which cudaMalloc is banned, a GPU whose memory is already claimed): the scratch is a 32 MiB
    array built into the library, so the problem must satisfy workspace_bytes(FN_COUNT, n_a, n_b) <=
    STATIC_SCRATCH_BYTES -- up to about 1.75 million intervals in B, any number of queries (else BitsError with status 9).  Pass `total_out` (int64[1], device) and this wrapper
    allocates nothing either.  One array per device: calls that overlap on the GPU race; calls on one stream do not."""
    n_a, n_b = a_start.numel(), b_start.numel()
    out = total_out if total_out is not None else torch.empty(1, dtype=torch.int64, device=a_start.device)
    _chk(lib().bits_count_static(_dev_u32(a_start, "a_start"), _dev_u32(a_end, "a_end"), n_a,
                                 _dev_u32(b_start, "b_start"), _dev_u32(b_end, "b_end"), n_b, flags,
                                 out.data_ptr(), _stream()))
    return out


def decide(a_start, a_end, b_start, b_end, flags: int = 0, workspace=None) -> torch.Tensor:
    """bits_decide -> device int32[1] tensor: 1 if some interval of A intersects one of B (valid after stream sync)."""
    dev = a_start.device
    n_a, n_b = a_start.numel(), b_start.numel()
    ws = _workspace(workspace_bytes(FN_COUNT, n_a, n_b, 0, 0, flags), workspace, dev)
    out = torch.empty(1, dtype=torch.int32, device=dev)
    _chk(lib().bits_decide(_dev_u32(a_start, "a_start"), _dev_u32(a_end, "a_end"), n_a,
                           _dev_u32(b_start, "b_start"), _dev_u32(b_end, "b_end"), n_b, flags,
                           ws.data_ptr(), ws.numel(), out.data_ptr(), _stream()))
    return out


def enumerate_pairs(a_start, a_end, b_start, b_end, flags: int = 0, workspace=None, capacity: int | None = None):
    """bits_enumerate -> (pair_a, pair_b, total): every intersecting pair as indices into A and B (device int32-typed
    uint32 tensors).  capacity = None: two calls, the first (capacity 0) sizes the outputs, `total` elements come
    back; synchronises once.  capacity = n: ONE call into arrays of n elements (no sort + count twice); pairs beyond n
    are not written, `total` is the full count either way."""
    dev = a_start.device
    n_a, n_b = a_start.numel(), b_start.numel()
    ws = _workspace(workspace_bytes(FN_ENUMERATE, n_a, n_b, 0, 0, flags), workspace, dev)
    total = torch.zeros(1, dtype=torch.int64, device=dev)
    args = (_dev_u32(a_start, "a_start"), _dev_u32(a_end, "a_end"), n_a, _dev_u32(b_start, "b_start"), _dev_u32(b_end, "b_end"), n_b,
            flags, ws.data_ptr(), ws.numel())
    if capacity is not None:
        pa = torch.empty(capacity, dtype=torch.int32, device=dev)
        pb = torch.empty(capacity, dtype=torch.int32, device=dev)
        _chk(lib().bits_enumerate(*args, pa.data_ptr() if capacity else 0, pb.data_ptr() if capacity else 0, capacity,
                                  total.data_ptr(), _stream()))
        return pa, pb, int(total.item())
    _chk(lib().bits_enumerate(*args, 0, 0, 0, total.data_ptr(), _stream()))
    n = int(total.item())
    pa = torch.empty(n, dtype=torch.int32, device=dev)
    pb = torch.empty(n, dtype=torch.int32, device=dev)
    if n:
        _chk(lib().bits_enumerate(*args, pa.data_ptr(), pb.data_ptr(), n, total.data_ptr(), _stream()))
    return pa, pb, n


def count_per_interval(a_start, a_end, b_start, b_end, flags: int = 0, workspace=None, counts_out=None,
                       total_out=None):
    """bits_count_per_interval -> (counts int32-typed uint32[n_a], total int64[1]) device tensors."""
    dev = a_start.device
    n_a, n_b = a_start.numel(), b_start.numel()
    ws = _workspace(workspace_bytes(FN_COUNT_PER_INTERVAL, n_a, n_b, 0, 0, flags), workspace, dev)
    counts = counts_out if counts_out is not None else torch.empty(n_a, dtype=torch.int32, device=dev)
    total = total_out if total_out is not None else torch.empty(1, dtype=torch.int64, device=dev)
    _chk(lib().bits_count_per_interval(_dev_u32(a_start, "a_start"), _dev_u32(a_end, "a_end"), n_a,
                                       _dev_u32(b_start, "b_start"), _dev_u32(b_end, "b_end"), n_b, flags,
                                       ws.data_ptr(), ws.numel(), _dev_u32(counts, "counts_out"),
                                       total.data_ptr(), _stream()))
    return counts, total


def mc_rounds(a_start, a_end, b_start, b_end, chrom_offsets, which: int, seed: int, round_begin: int,
              n_rounds: int, flags: int = 0, workspace=None, observed_out=None, round_counts_out=None):
    """bits_mc_rounds -> (observed int64[1], round_counts int64[n_rounds]) device tensors."""
    dev = a_start.device
    off = _offsets(chrom_offsets)
    n_a, n_b = a_start.numel(), b_start.numel()
    ws = _workspace(workspace_bytes(FN_MC_ROUNDS, n_a, n_b, off.size - 1, which, flags), workspace, dev)
    obs = observed_out if observed_out is not None else torch.empty(1, dtype=torch.int64, device=dev)
    rc = round_counts_out if round_counts_out is not None else torch.empty(n_rounds, dtype=torch.int64, device=dev)
    _chk(lib().bits_mc_rounds(_dev_u32(a_start, "a_start"), _dev_u32(a_end, "a_end"), n_a,
                              _dev_u32(b_start, "b_start"), _dev_u32(b_end, "b_end"), n_b,
                              off.ctypes.data, off.size - 1, which, seed, round_begin, n_rounds, flags,
                              ws.data_ptr(), ws.numel(), obs.data_ptr(), rc.data_ptr() if n_rounds else 0, _stream()))
    return obs, rc


def place(spans, chrom_offsets, seed: int, rnd: int, tag: int, workspace=None):
    """bits_place -> (start, end) device tensors for one round."""
    dev = spans.device
    off = _offsets(chrom_offsets)
    n = spans.numel()
    ws = _workspace(workspace_bytes(FN_PLACE, 0, 0, off.size - 1), workspace, dev)
    s = torch.empty(n, dtype=torch.int32, device=dev)
    e = torch.empty(n, dtype=torch.int32, device=dev)
    _chk(lib().bits_place(_dev_u32(spans, "spans"), n, off.ctypes.data, off.size - 1, seed, rnd, tag,
                          ws.data_ptr(), ws.numel(), _dev_u32(s, "start_out"), _dev_u32(e, "end_out"), _stream()))
    return s, e


def sort_u32(keys, workspace=None) -> torch.Tensor:
    """bits_sort_u32 -> ascending copy of a 32-bit key tensor (compared as unsigned)."""
    dev = keys.device
    n = keys.numel()
    ws = _workspace(workspace_bytes(FN_SORT, 0, n), workspace, dev)
    out = torch.empty_like(keys)
    _chk(lib().bits_sort_u32(_dev_u32(keys, "keys_in"), _dev_u32(out, "keys_out"), n, ws.data_ptr(), ws.numel(),
                             _stream()))
    return out


# --------------------------------------------------------------------------------------------
@dataclass
class McResult:
    observed: int
    round_counts: np.ndarray      # uint64[n_rounds]
    p_enrich: float
    p_deplete: float


def pvalue(observed: int, round_counts, tail: int = 0) -> float:
    rc = np.ascontiguousarray(round_counts, dtype=np.uint64)
    return float(lib().bits_pvalue(int(observed), rc.ctypes.data if rc.size else 0, rc.size, tail))


def enrichment(observed: int, round_counts) -> float:
    """bits_enrichment: log2(observed / median of the round counts)."""
    rc = np.ascontiguousarray(round_counts, dtype=np.uint64)
    return float(lib().bits_enrichment(int(observed), rc.ctypes.data if rc.size else 0, rc.size))


def screen_concat(starts, ends, track_offsets, chrom_offsets, seed: int, n_rounds: int, round_begin: int = 0,
                  flags: int = 0, workspace=None, observed_out=None, round_counts_out=None):
    """bits_screen on K tracks passed concatenated (device uint32 tensors + host offsets uint64[K + 1]) ->
    (observed int64[K, K], round_counts int64[K, K, n_rounds]) device tensors, valid after stream sync."""
    dev = starts.device
    toff = np.ascontiguousarray(track_offsets, dtype=np.uint64)
    K = toff.size - 1
    off = _offsets(chrom_offsets)
    nbytes = int(lib().bits_screen_workspace_bytes(toff.ctypes.data, K, off.size - 1))
    if nbytes == 0:
        raise BitsError(2, "bad track offset table")
    ws = _workspace(nbytes, workspace, dev)
    obs = observed_out if observed_out is not None else torch.empty((K, K), dtype=torch.int64, device=dev)
    rc = round_counts_out if round_counts_out is not None else torch.empty((K, K, n_rounds), dtype=torch.int64, device=dev)
    _chk(lib().bits_screen(_dev_u32(starts, "starts"), _dev_u32(ends, "ends"), toff.ctypes.data, K, off.ctypes.data,
                           off.size - 1, seed, round_begin, n_rounds, flags, ws.data_ptr(), ws.numel(), obs.data_ptr(),
                           rc.data_ptr() if n_rounds else 0, _stream()))
    return obs, rc


def screen_enrichment(observed, round_counts) -> np.ndarray:
    """bits_screen_enrichment on host arrays: log2(observed / median of the pair's round counts), shape of `observed`."""
    o = np.ascontiguousarray(observed, dtype=np.uint64)
    r = np.ascontiguousarray(round_counts, dtype=np.uint64)
    n_rounds = r.size // o.size if o.size else 0
    out = np.empty(o.shape, dtype=np.float64)
    _chk(lib().bits_screen_enrichment(o.ctypes.data, r.ctypes.data if r.size else 0, o.size, n_rounds, out.ctypes.data))
    return out


def screen(tracks, chrom_offsets, seed: int, n_rounds: int, round_begin: int = 0):
    """The paper's co-localisation screen (Fig. 3) over K interval sets, `tracks` = [(start, end)
    device tensors]: one bits_screen call (every track sorted and indexed once, all pairs and rounds in gridded
    launches, pair id in the Philox counter).  Returns numpy arrays (observed uint64[K, K], enrichment
    float64[K, K], round_counts uint64[K, K, n_rounds]).  Marshalling only: the tracks are concatenated for the call."""
    K = len(tracks)
    toff = np.zeros(K + 1, dtype=np.uint64)
    toff[1:] = np.cumsum([t[0].numel() for t in tracks])
    starts = torch.cat([t[0] for t in tracks]) if K > 1 else tracks[0][0]
    ends = torch.cat([t[1] for t in tracks]) if K > 1 else tracks[0][1]
    obs, rc = screen_concat(starts, ends, toff, chrom_offsets, seed, n_rounds, round_begin)
    torch.cuda.synchronize(starts.device)
    obs_h = obs.cpu().numpy().view(np.uint64)
    rc_h = rc.cpu().numpy().view(np.uint64)
    return obs_h, screen_enrichment(obs_h, rc_h), rc_h


def host_workspace(fn: int, n_a: int, n_b: int, n_chrom: int = 0, which: int = 0, n_rounds: int = 0,
                   device="cuda:0", flags: int = 0) -> torch.Tensor:
    """Device workspace big enough for the *_host variant of `fn`."""
    nbytes = workspace_bytes(fn, n_a, n_b, n_chrom, which, flags) + host_staging_bytes(fn, n_a, n_b, n_rounds)
    return torch.empty(max(nbytes, 256), dtype=torch.uint8, device=device)


def count_host(a_start, a_end, b_start, b_end, flags: int = 0, workspace=None, device="cuda:0") -> int:
    a_s, a_e, b_s, b_e = (_host_u32(x, n) for x, n in ((a_start, "a_start"), (a_end, "a_end"),
                                                        (b_start, "b_start"), (b_end, "b_end")))
    ws = workspace if workspace is not None else host_workspace(FN_COUNT, a_s.size, b_s.size, device=device)
    total = np.zeros(1, dtype=np.uint64)
    with torch.cuda.device(ws.device):
        _chk(lib().bits_count_host(a_s.ctypes.data, a_e.ctypes.data, a_s.size, b_s.ctypes.data, b_e.ctypes.data,
                                   b_s.size, flags, ws.data_ptr(), ws.numel(), total.ctypes.data, _stream()))
    return int(total[0])


def count_per_interval_host(a_start, a_end, b_start, b_end, flags: int = 0, workspace=None, device="cuda:0",
                            counts_out=None):
    a_s, a_e, b_s, b_e = (_host_u32(x, n) for x, n in ((a_start, "a_start"), (a_end, "a_end"),
                                                        (b_start, "b_start"), (b_end, "b_end")))
    ws = workspace if workspace is not None else host_workspace(FN_COUNT_PER_INTERVAL, a_s.size, b_s.size,
                                                                device=device)
    counts = counts_out if counts_out is not None else np.zeros(a_s.size, dtype=np.uint32)
    total = np.zeros(1, dtype=np.uint64)
    with torch.cuda.device(ws.device):
        _chk(lib().bits_count_per_interval_host(a_s.ctypes.data, a_e.ctypes.data, a_s.size, b_s.ctypes.data,
                                                b_e.ctypes.data, b_s.size, flags, ws.data_ptr(), ws.numel(),
                                                counts.ctypes.data if a_s.size else 0, total.ctypes.data, _stream()))
    return counts, int(total[0])


def mc_rounds_host(a_start, a_end, b_start, b_end, chrom_offsets, which: int, seed: int, round_begin: int,
                   n_rounds: int, flags: int = 0, workspace=None, device="cuda:0", round_counts_out=None) -> McResult:
    a_s, a_e, b_s, b_e = (_host_u32(x, n) for x, n in ((a_start, "a_start"), (a_end, "a_end"),
                                                        (b_start, "b_start"), (b_end, "b_end")))
    off = _offsets(chrom_offsets)
    ws = workspace if workspace is not None else host_workspace(FN_MC_ROUNDS, a_s.size, b_s.size, off.size - 1,
                                                                which, n_rounds, device=device)
    obs = np.zeros(1, dtype=np.uint64)
    rc = round_counts_out if round_counts_out is not None else np.zeros(n_rounds, dtype=np.uint64)
    with torch.cuda.device(ws.device):
        _chk(lib().bits_mc_rounds_host(a_s.ctypes.data, a_e.ctypes.data, a_s.size, b_s.ctypes.data, b_e.ctypes.data,
                                       b_s.size, off.ctypes.data, off.size - 1, which, seed, round_begin, n_rounds,
                                       flags, ws.data_ptr(), ws.numel(), obs.ctypes.data,
                                       rc.ctypes.data if n_rounds else 0, _stream()))
    o = int(obs[0])
    return McResult(o, rc, pvalue(o, rc, 0), pvalue(o, rc, 1))
