"""Thin ctypes binding of include/gene_nl.h -- same names, argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libgene_nl.so.  PyTorch appears only as the
owner of device memory and streams (tensor.data_ptr(), torch.cuda.current_stream()).  If the shared
library is missing it is built in-tree with nvcc; if that fails, or no CUDA device is present at
gene_nl_create time, the call raises -- there is no CPU fallback.
"""
from __future__ import annotations

import ctypes
import os
import threading

from . import build as _build

GENE_NL_OK, GENE_NL_EINVAL, GENE_NL_EUNSUPPORTED, GENE_NL_ECUDA, GENE_NL_ENOMEM = 0, 1, 2, 3, 4

# every symbol include/gene_nl.h declares (the product boundary) ...
EXPORTED_SYMBOLS = (
    "gene_nl_create", "gene_nl_compute", "gene_nl_compute_em", "gene_nl_compute_host", "gene_nl_compute_em_host",
    "gene_nl_destroy", "gene_nl_last_error", "gene_nl_set_scratch_bytes", "gene_nl_set_plane_kernel",
    "gene_nl_workspace_bytes", "gene_nl_launches_per_compute", "gene_nl_query", "gene_nl_compute_static",
    "gene_nlx_create", "gene_nlx_compute", "gene_nlx_compute_host", "gene_nlx_destroy", "gene_nlx_query",
)
# ... and include/gene_nl_bench.h (benchmark-only helpers, not on the hot path)
BENCH_SYMBOLS = ("gene_nl_compute_profiled", "gene_nl_probe_peaks")

_lock = threading.Lock()
_lib = None


class GeneNLError(RuntimeError):
    pass


def library_path() -> str:
    return _build.LIB


def load_library() -> ctypes.CDLL:
    """Load (building first if needed) paper_1310_1485_b200/libgene_nl.so and declare prototypes."""
    global _lib
    with _lock:
        if _lib is not None:
            return _lib
        path = _build.build()
        if not os.path.exists(path):
            raise GeneNLError(f"CUDA extension {path} is missing and could not be built")
        lib = ctypes.CDLL(path)
        vp, dbl, i = ctypes.c_void_p, ctypes.c_double, ctypes.c_int
        lib.gene_nl_create.argtypes = [i, i, i, i, i, i, dbl, dbl, i]
        lib.gene_nl_create.restype = vp
        lib.gene_nl_compute.argtypes = [vp, vp, vp, vp, dbl, vp]
        lib.gene_nl_compute.restype = i
        lib.gene_nl_compute_em.argtypes = [vp, vp, vp, ctypes.POINTER(dbl), vp, vp, dbl, vp]
        lib.gene_nl_compute_em.restype = i
        lib.gene_nl_compute_profiled.argtypes = [vp, vp, vp, vp, dbl, vp, ctypes.POINTER(dbl), ctypes.POINTER(i)]
        lib.gene_nl_compute_profiled.restype = i
        lib.gene_nl_compute_host.argtypes = [vp, vp, vp, vp, dbl]
        lib.gene_nl_compute_host.restype = i
        lib.gene_nl_compute_em_host.argtypes = [vp, vp, vp, ctypes.POINTER(dbl), vp, vp, dbl]
        lib.gene_nl_compute_em_host.restype = i
        lib.gene_nl_set_scratch_bytes.argtypes = [vp, ctypes.c_size_t]
        lib.gene_nl_set_scratch_bytes.restype = i
        lib.gene_nl_set_plane_kernel.argtypes = [vp, i]
        lib.gene_nl_set_plane_kernel.restype = i
        lib.gene_nl_destroy.argtypes = [vp]
        lib.gene_nl_destroy.restype = None
        lib.gene_nl_last_error.argtypes = []
        lib.gene_nl_last_error.restype = ctypes.c_char_p
        lib.gene_nl_workspace_bytes.argtypes = [vp]
        lib.gene_nl_workspace_bytes.restype = ctypes.c_size_t
        lib.gene_nl_launches_per_compute.argtypes = [vp]
        lib.gene_nl_launches_per_compute.restype = i
        lib.gene_nl_query.argtypes = [vp, i]
        lib.gene_nl_query.restype = dbl
        lib.gene_nl_compute_static.argtypes = [i, i, i, i, i, i, dbl, dbl, vp, vp, vp, dbl, vp]
        lib.gene_nl_compute_static.restype = i
        lib.gene_nl_probe_peaks.argtypes = [ctypes.POINTER(dbl)]
        lib.gene_nl_probe_peaks.restype = i
        ll = ctypes.c_longlong
        lib.gene_nlx_create.argtypes = [i, i, ll]
        lib.gene_nlx_create.restype = vp
        lib.gene_nlx_compute.argtypes = [vp, vp, vp, vp, vp, vp, vp, dbl, vp]
        lib.gene_nlx_compute.restype = i
        lib.gene_nlx_compute_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, dbl]
        lib.gene_nlx_compute_host.restype = i
        lib.gene_nlx_destroy.argtypes = [vp]
        lib.gene_nlx_destroy.restype = None
        lib.gene_nlx_query.argtypes = [vp, i]
        lib.gene_nlx_query.restype = dbl
        _lib = lib
        return lib


def gene_nl_last_error() -> str:
    return load_library().gene_nl_last_error().decode()


def gene_nl_create(nx0, nky0, nz, nv, nw, nspec, kxmin, kymin, chi_has_v) -> int:
    """Returns the opaque plan handle (an integer address); raises GeneNLError on failure."""
    h = load_library().gene_nl_create(int(nx0), int(nky0), int(nz), int(nv), int(nw), int(nspec),
                                      float(kxmin), float(kymin), int(chi_has_v))  # 0, 1 or GENE_NL_CHI_EM
    if not h:
        raise GeneNLError(gene_nl_last_error() or "gene_nl_create failed")
    return h


def _ptr(x) -> int:
    return x.data_ptr() if hasattr(x, "data_ptr") else int(x)


def gene_nl_compute(h, chi, g, rhs, scale, stream=None) -> None:
    """rhs += scale*N(chi, g) on DEVICE arrays (torch CUDA tensors or raw device addresses).

    Asynchronous on `stream` (a torch.cuda.Stream, a raw cudaStream_t address, or None for torch's
    current stream)."""
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    elif hasattr(stream, "cuda_stream"):
        stream = stream.cuda_stream
    rc = load_library().gene_nl_compute(h, _ptr(chi), _ptr(g), _ptr(rhs), float(scale), int(stream) or None)
    if rc != GENE_NL_OK:
        raise GeneNLError(f"gene_nl_compute failed ({rc}): {gene_nl_last_error()}")


GENE_NL_CHI_EM = 2
GENE_NL_STATIC_NX0, GENE_NL_STATIC_NKY0, GENE_NL_STATIC_MAX_GROUPS = 96, 48, 64


def gene_nl_compute_static(nx0, nky0, nz, nv, nw, nspec, kxmin, kymin, chi, g, rhs, scale, stream=None) -> None:
    """rhs += scale*N(chi, g) with chi shaped like g, for callers that must not allocate device memory.

    No plan: the library's other entry points cudaMalloc their tables and scratch, which a caller whose own pool
    already owns the whole device, or whose other streams must not be stalled by cudaMalloc's device-wide
    synchronisation, cannot afford.  This one keeps the planes in flight in a static device array inside the library
    (33.75 MiB, held by every GPU that loads it) and supports planes of 96 x 48 modes only; anything else raises.
    Calls on one device share that array: do not let two of them overlap on the GPU.  The first call per device
    does a synchronous set-up (keep it outside stream capture).  See include/gene_nl.h."""
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    elif hasattr(stream, "cuda_stream"):
        stream = stream.cuda_stream
    rc = load_library().gene_nl_compute_static(int(nx0), int(nky0), int(nz), int(nv), int(nw), int(nspec), float(kxmin),
                                               float(kymin), _ptr(chi), _ptr(g), _ptr(rhs), float(scale),
                                               int(stream) or None)
    if rc != GENE_NL_OK:
        raise GeneNLError(f"gene_nl_compute_static failed ({rc}): {gene_nl_last_error()}")


def gene_nl_compute_em(h, phi, apar, vpar, g, rhs, scale, stream=None) -> None:
    """rhs += scale*N(phi - vpar*apar, g) with chi composed on the device; vpar: nv*nspec floats (host)."""
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    elif hasattr(stream, "cuda_stream"):
        stream = stream.cuda_stream
    vals = [float(x) for x in vpar]
    arr = (ctypes.c_double * len(vals))(*vals)
    rc = load_library().gene_nl_compute_em(h, _ptr(phi), _ptr(apar), arr, _ptr(g), _ptr(rhs), float(scale),
                                           int(stream) or None)
    if rc != GENE_NL_OK:
        raise GeneNLError(f"gene_nl_compute_em failed ({rc}): {gene_nl_last_error()}")


def gene_nl_compute_em_host(h, phi, apar, vpar, g, rhs, scale) -> None:
    """gene_nl_compute_em on HOST arrays (torch CPU tensors, ideally pinned, or raw addresses); synchronous."""
    vals = [float(x) for x in vpar]
    arr = (ctypes.c_double * len(vals))(*vals)
    rc = load_library().gene_nl_compute_em_host(h, _ptr(phi), _ptr(apar), arr, _ptr(g), _ptr(rhs), float(scale))
    if rc != GENE_NL_OK:
        raise GeneNLError(f"gene_nl_compute_em_host failed ({rc}): {gene_nl_last_error()}")


def gene_nl_set_scratch_bytes(h, nbytes: int) -> None:
    """Change the plan's scratch budget (bytes per scratch set); more, smaller batches -- never a different result."""
    rc = load_library().gene_nl_set_scratch_bytes(h, int(nbytes))
    if rc != GENE_NL_OK:
        raise GeneNLError(f"gene_nl_set_scratch_bytes failed ({rc}): {gene_nl_last_error()}")


GENE_NL_KERNEL_AUTO, GENE_NL_KERNEL_CLUSTER, GENE_NL_KERNEL_GROUP, GENE_NL_KERNEL_BATCHED, GENE_NL_KERNEL_WARP = 0, 1, 2, 3, 4


def gene_nl_set_plane_kernel(h, kind: int) -> None:
    """Kernel family for the g side of a plane: GENE_NL_KERNEL_AUTO, _GROUP (384 x 192, 768 x 384, 144 x 144 padded
    grids), _WARP (the same grids, not EM), _CLUSTER (384 x 192) or _BATCHED (any size); see include/gene_nl.h."""
    rc = load_library().gene_nl_set_plane_kernel(h, int(kind))
    if rc != GENE_NL_OK:
        raise GeneNLError(f"gene_nl_set_plane_kernel failed ({rc}): {gene_nl_last_error()}")


KERNEL_CLASSES = ("k_xinv", "k_yreal", "k_ybracket", "k_xfwd", "k_plane_fused")


def gene_nl_compute_profiled(h, chi, g, rhs, scale, stream=None):
    """gene_nl_compute with per-launch CUDA events; returns ({class: ms}, {class: launches}); synchronises."""
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    elif hasattr(stream, "cuda_stream"):
        stream = stream.cuda_stream
    ms = (ctypes.c_double * len(KERNEL_CLASSES))()
    n = (ctypes.c_int * len(KERNEL_CLASSES))()
    rc = load_library().gene_nl_compute_profiled(h, _ptr(chi), _ptr(g), _ptr(rhs), float(scale),
                                                 int(stream) or None, ms, n)
    if rc != GENE_NL_OK:
        raise GeneNLError(f"gene_nl_compute_profiled failed ({rc}): {gene_nl_last_error()}")
    return dict(zip(KERNEL_CLASSES, map(float, ms))), dict(zip(KERNEL_CLASSES, map(int, n)))


def gene_nl_compute_host(h, chi, g, rhs, scale) -> None:
    """Same on HOST arrays (torch CPU tensors, ideally pinned, or raw addresses); synchronous."""
    rc = load_library().gene_nl_compute_host(h, _ptr(chi), _ptr(g), _ptr(rhs), float(scale))
    if rc != GENE_NL_OK:
        raise GeneNLError(f"gene_nl_compute_host failed ({rc}): {gene_nl_last_error()}")


def gene_nl_destroy(h) -> None:
    if h:
        load_library().gene_nl_destroy(h)


def gene_nl_workspace_bytes(h) -> int:
    return int(load_library().gene_nl_workspace_bytes(h))


def gene_nl_launches_per_compute(h) -> int:
    return int(load_library().gene_nl_launches_per_compute(h))


def gene_nl_query(h, what: int) -> float:
    return float(load_library().gene_nl_query(h, int(what)))


def gene_nl_probe_peaks():
    """(FP64 TFLOP/s, shared-memory GB/s, SM clock MHz) measured on the current device."""
    out = (ctypes.c_double * 3)()
    rc = load_library().gene_nl_probe_peaks(out)
    if rc != GENE_NL_OK:
        raise GeneNLError(f"gene_nl_probe_peaks failed ({rc})")
    return float(out[0]), float(out[1]), float(out[2])


# ---- x-global variant (include/gene_nl.h, gene_nlx_*) ----
def gene_nlx_create(nx, nky0, planes) -> int:
    h = load_library().gene_nlx_create(int(nx), int(nky0), int(planes))
    if not h:
        raise GeneNLError(gene_nl_last_error() or "gene_nlx_create failed")
    return h


def gene_nlx_compute(h, vex, vey, dxg, dyg, pref, rhs, scale, stream=None) -> None:
    """rhs += scale*pref[x]*N^ on DEVICE arrays (torch CUDA tensors or raw addresses); asynchronous on `stream`."""
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    elif hasattr(stream, "cuda_stream"):
        stream = stream.cuda_stream
    rc = load_library().gene_nlx_compute(h, _ptr(vex), _ptr(vey), _ptr(dxg), _ptr(dyg), _ptr(pref), _ptr(rhs),
                                         float(scale), int(stream) or None)
    if rc != GENE_NL_OK:
        raise GeneNLError(f"gene_nlx_compute failed ({rc}): {gene_nl_last_error()}")


def gene_nlx_compute_host(h, vex, vey, dxg, dyg, pref, rhs, scale) -> None:
    """Same on HOST arrays (torch CPU tensors, ideally pinned, or raw addresses), chunked over CUDA streams; synchronous."""
    rc = load_library().gene_nlx_compute_host(h, _ptr(vex), _ptr(vey), _ptr(dxg), _ptr(dyg), _ptr(pref), _ptr(rhs),
                                              float(scale))
    if rc != GENE_NL_OK:
        raise GeneNLError(f"gene_nlx_compute_host failed ({rc}): {gene_nl_last_error()}")


def gene_nlx_destroy(h) -> None:
    if h:
        load_library().gene_nlx_destroy(h)


def gene_nlx_query(h, what: int) -> float:
    return float(load_library().gene_nlx_query(h, int(what)))


class GeneNL:
    """Context-manager convenience around create/compute/destroy for a workloads.Workload."""

    def __init__(self, wl, scratch_bytes=None, plane_kernel=None):
        self.wl = wl
        self.h = gene_nl_create(wl.nx0, wl.nky0, wl.nz, wl.nv, wl.nw, wl.nspec, wl.kxmin, wl.kymin, wl.chi_has_v)
        if plane_kernel is not None:
            gene_nl_set_plane_kernel(self.h, plane_kernel)
        if scratch_bytes is not None:
            gene_nl_set_scratch_bytes(self.h, scratch_bytes)

    def compute(self, chi, g, rhs, scale=None, stream=None):
        gene_nl_compute(self.h, chi, g, rhs, self.wl.scale if scale is None else scale, stream)

    def compute_profiled(self, chi, g, rhs, scale=None, stream=None):
        return gene_nl_compute_profiled(self.h, chi, g, rhs, self.wl.scale if scale is None else scale, stream)

    def compute_host(self, chi, g, rhs, scale=None):
        gene_nl_compute_host(self.h, chi, g, rhs, self.wl.scale if scale is None else scale)

    def query(self, what):
        return gene_nl_query(self.h, what)

    @property
    def launches_per_compute(self):
        return gene_nl_launches_per_compute(self.h)

    @property
    def workspace_bytes(self):
        return gene_nl_workspace_bytes(self.h)

    def close(self):
        if self.h:
            gene_nl_destroy(self.h)
            self.h = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
