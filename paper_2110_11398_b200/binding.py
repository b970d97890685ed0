"""Thin ctypes binding of ``include/nf.h`` -- argument marshalling only.

Every step of the hot path (cell ids, histogram, prefix sums, stable sort, gather, scheduling,
direct sum, scatter) runs in the CUDA kernels of ``libnf_b200.so``; torch is used for device
memory, streams and nothing else.  The functions carry the C names (``nf_plan_create``,
``nf_bin``, ``nf_accel``, ``nf_destroy``, ...); ``Plan`` is a convenience wrapper around them.

There is no CPU fallback: if the library cannot be loaded, importing this module raises.
Operation defined in PAPER.md:337-349 (sec. 3.1); see ``include/nf.h``.
"""
from __future__ import annotations

import ctypes
import os

import torch

from . import build as _build

NF_OK, NF_ERR_ARG, NF_ERR_DOMAIN, NF_ERR_STATE, NF_ERR_NOMEM, NF_ERR_CUDA = 0, -1, -2, -3, -4, -5
_ERR_NAMES = {-1: "NF_ERR_ARG", -2: "NF_ERR_DOMAIN", -3: "NF_ERR_STATE", -4: "NF_ERR_NOMEM", -5: "NF_ERR_CUDA"}

EXPORTS = [
    "nf_plan_create", "nf_bin", "nf_rebin", "nf_accel", "nf_accel_density", "nf_accel_kick", "nf_set_masses", "nf_set_sink_slabs", "nf_destroy", "nf_bin_host", "nf_accel_host",
    "nf_last_error", "nf_set_stream", "nf_workspace_bytes", "nf_set_workspace", "nf_get_binning",
    "nf_get_layout", "nf_get_stats", "nf_set_option",
    "nf_slab_histogram", "nf_slab_select", "nf_get_slab_cost", "nf_slab_partition", "nf_slab_histogram_static",
]


class NFError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{_ERR_NAMES.get(code, code)}: {msg}")
        self.code = code


class nf_stats(ctypes.Structure):
    _fields_ = [
        ("n", ctypes.c_longlong), ("cells", ctypes.c_longlong), ("padded_slots", ctypes.c_longlong),
        ("units", ctypes.c_longlong), ("interactions", ctypes.c_longlong),
        ("ms_bin", ctypes.c_float), ("ms_accel", ctypes.c_float),
        ("sm_count", ctypes.c_int), ("clock_khz", ctypes.c_int),
        ("accel_grid", ctypes.c_int), ("accel_block", ctypes.c_int),
        ("kernel_launches_bin", ctypes.c_int), ("kernel_launches_accel", ctypes.c_int),
        ("rebin_path", ctypes.c_int), ("rebin_movers", ctypes.c_longlong),
    ]


def _load() -> ctypes.CDLL:
    path = _build.LIB
    if not os.path.exists(path) or _build.stale():
        try:
            _build.build()
        except Exception as e:  # no nvcc on this box and no prebuilt library: fail loudly
            if not os.path.exists(path):
                raise ImportError(f"libnf_b200.so is missing and could not be built ({e}); "
                                  "there is no CPU fallback") from e
            import warnings
            warnings.warn(f"libnf_b200.so is older than its sources and the rebuild failed ({e}): running the STALE library",
                          RuntimeWarning)
    lib = ctypes.CDLL(path)
    vp, ll, i32, dbl = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int, ctypes.c_double
    pp = ctypes.POINTER(ctypes.c_void_p)
    lib.nf_plan_create.restype = vp
    lib.nf_plan_create.argtypes = [i32, dbl, dbl, i32]
    lib.nf_bin.restype = i32
    lib.nf_bin.argtypes = [vp, vp, ll]
    lib.nf_rebin.restype = i32
    lib.nf_rebin.argtypes = [vp, vp]
    lib.nf_accel.restype = i32
    lib.nf_accel.argtypes = [vp, vp]
    lib.nf_accel_density.restype = i32
    lib.nf_accel_density.argtypes = [vp, vp, vp, dbl]
    lib.nf_accel_kick.restype = i32
    lib.nf_accel_kick.argtypes = [vp, vp, vp, dbl, vp]
    lib.nf_set_masses.restype = i32
    lib.nf_set_masses.argtypes = [vp, vp]
    lib.nf_set_sink_slabs.restype = i32
    lib.nf_set_sink_slabs.argtypes = [vp, i32, i32]
    lib.nf_destroy.restype = None
    lib.nf_destroy.argtypes = [vp]
    lib.nf_bin_host.restype = i32
    lib.nf_bin_host.argtypes = [vp, vp, ll]
    lib.nf_accel_host.restype = i32
    lib.nf_accel_host.argtypes = [vp, vp]
    lib.nf_last_error.restype = ctypes.c_char_p
    lib.nf_last_error.argtypes = []
    lib.nf_set_stream.restype = i32
    lib.nf_set_stream.argtypes = [vp, vp]
    lib.nf_workspace_bytes.restype = ctypes.c_size_t
    lib.nf_workspace_bytes.argtypes = [vp, ll]
    lib.nf_set_workspace.restype = i32
    lib.nf_set_workspace.argtypes = [vp, vp, ctypes.c_size_t]
    lib.nf_get_binning.restype = i32
    lib.nf_get_binning.argtypes = [vp, pp, pp, pp, pp]
    lib.nf_get_layout.restype = i32
    lib.nf_get_layout.argtypes = [vp, pp, pp, pp, pp, ctypes.POINTER(dbl)]
    lib.nf_get_stats.restype = i32
    lib.nf_get_stats.argtypes = [vp, ctypes.POINTER(nf_stats)]
    lib.nf_set_option.restype = i32
    lib.nf_set_option.argtypes = [vp, ctypes.c_char_p, ll]
    lib.nf_slab_histogram.restype = i32
    lib.nf_slab_histogram.argtypes = [vp, vp, ll, ctypes.POINTER(ll)]
    lib.nf_slab_histogram_static.restype = i32
    lib.nf_slab_histogram_static.argtypes = [vp, vp, ll, ctypes.POINTER(ll)]
    lib.nf_slab_select.restype = i32
    lib.nf_slab_select.argtypes = [vp, vp, ll, i32, i32, vp, vp, ll, ctypes.POINTER(ll)]
    lib.nf_get_slab_cost.restype = i32
    lib.nf_get_slab_cost.argtypes = [vp, ctypes.POINTER(dbl)]
    lib.nf_slab_partition.restype = i32
    lib.nf_slab_partition.argtypes = [ctypes.POINTER(dbl), i32, i32, ctypes.POINTER(i32), ctypes.POINTER(i32)]
    return lib


_lib = _load()
LIB_PATH = _build.LIB


def nf_last_error() -> str:
    return (_lib.nf_last_error() or b"").decode()


def _check(rc: int):
    if rc != NF_OK:
        raise NFError(rc, nf_last_error())


def _dev_f32(t: torch.Tensor, what: str) -> torch.Tensor:
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
            and t.dim() == 2 and t.shape[1] == 3):
        raise TypeError(f"{what} must be a contiguous CUDA float32 tensor of shape [n, 3]")
    return t


def _host_f32(t: torch.Tensor, what: str) -> torch.Tensor:
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
            and t.dim() == 2 and t.shape[1] == 3):
        raise TypeError(f"{what} must be a contiguous CPU float32 tensor of shape [n, 3]")
    return t


# ---- the C calls, same names ------------------------------------------------------------------
# The C ABI takes bare pointers: a caller buffer shorter than the n of the last binning would be written out of bounds
# on the device.  The binding therefore remembers (n, cpd^3) per plan handle and checks every output tensor against it.
_SHAPE: dict[int, list] = {}


def _rows(plan: int, t: torch.Tensor, what: str) -> None:
    n = _SHAPE.get(plan, [None, None])[0]
    if n is not None and t.shape[0] != n:
        raise ValueError(f"{what} has {t.shape[0]} rows but the plan last binned {n} particles")


def nf_plan_create(cpd: int, L: float, eps: float, R: int = 2) -> int:
    h = _lib.nf_plan_create(int(cpd), float(L), float(eps), int(R))
    if not h:
        raise NFError(NF_ERR_ARG, nf_last_error())
    _SHAPE[h] = [None, int(cpd) ** 3]
    return h


def nf_destroy(plan: int) -> None:
    _SHAPE.pop(plan, None)
    _lib.nf_destroy(plan)


def nf_set_stream(plan: int, cuda_stream: int) -> None:
    _check(_lib.nf_set_stream(plan, ctypes.c_void_p(cuda_stream)))


def nf_bin(plan: int, pos: torch.Tensor) -> None:
    pos = _dev_f32(pos, "pos")
    if plan in _SHAPE:
        _SHAPE[plan][0] = None
    _check(_lib.nf_bin(plan, ctypes.c_void_p(pos.data_ptr()), pos.shape[0]))
    if plan in _SHAPE:
        _SHAPE[plan][0] = pos.shape[0]


def nf_rebin(plan: int, pos: torch.Tensor) -> None:
    """The same particles after they moved: new positions in the same input order (include/nf.h)."""
    pos = _dev_f32(pos, "pos")
    _rows(plan, pos, "pos")
    _check(_lib.nf_rebin(plan, ctypes.c_void_p(pos.data_ptr())))


def nf_accel(plan: int, acc: torch.Tensor) -> None:
    acc = _dev_f32(acc, "acc")
    _rows(plan, acc, "acc")
    _check(_lib.nf_accel(plan, ctypes.c_void_p(acc.data_ptr())))


def nf_accel_density(plan: int, acc: torch.Tensor, rho: torch.Tensor, b: float) -> None:
    acc = _dev_f32(acc, "acc")
    if not (isinstance(rho, torch.Tensor) and rho.is_cuda and rho.dtype == torch.float32 and rho.is_contiguous()
            and rho.dim() == 1 and rho.shape[0] == acc.shape[0]):
        raise TypeError("rho must be a contiguous CUDA float32 tensor of shape [n]")
    _rows(plan, acc, "acc")
    _check(_lib.nf_accel_density(plan, ctypes.c_void_p(acc.data_ptr()), ctypes.c_void_p(rho.data_ptr()), float(b)))


def nf_accel_kick(plan: int, acc: torch.Tensor | None, vel: torch.Tensor | None, dt: float,
                  amax_cell: torch.Tensor | None) -> None:
    pa = ctypes.c_void_p(_dev_f32(acc, "acc").data_ptr()) if acc is not None else None
    pv = ctypes.c_void_p(_dev_f32(vel, "vel").data_ptr()) if vel is not None else None
    pm = None
    for t, what in ((acc, "acc"), (vel, "vel")):
        if t is not None:
            _rows(plan, t, what)
    if amax_cell is not None:
        if not (amax_cell.is_cuda and amax_cell.dtype == torch.float32 and amax_cell.is_contiguous() and amax_cell.dim() == 1):
            raise TypeError("amax_cell must be a contiguous CUDA float32 tensor of shape [cpd^3]")
        nc = _SHAPE.get(plan, [None, None])[1]
        if nc is not None and amax_cell.shape[0] != nc:
            raise ValueError(f"amax_cell has {amax_cell.shape[0]} entries but the plan has {nc} cells")
        pm = ctypes.c_void_p(amax_cell.data_ptr())
    _check(_lib.nf_accel_kick(plan, pa, pv, float(dt), pm))


def nf_set_masses(plan: int, mass: torch.Tensor | None, n: int) -> None:
    if mass is None:
        _check(_lib.nf_set_masses(plan, None))
        return
    if not (mass.is_cuda and mass.dtype == torch.float32 and mass.is_contiguous() and mass.shape == (n,)):
        raise TypeError("mass must be a contiguous CUDA float32 tensor of shape [n]")
    _check(_lib.nf_set_masses(plan, ctypes.c_void_p(mass.data_ptr())))


def nf_set_sink_slabs(plan: int, x_first: int, n_slabs: int) -> None:
    _check(_lib.nf_set_sink_slabs(plan, int(x_first), int(n_slabs)))


def nf_bin_host(plan: int, pos_host: torch.Tensor) -> None:
    pos_host = _host_f32(pos_host, "pos_host")
    if plan in _SHAPE:
        _SHAPE[plan][0] = None
    _check(_lib.nf_bin_host(plan, ctypes.c_void_p(pos_host.data_ptr()), pos_host.shape[0]))
    if plan in _SHAPE:
        _SHAPE[plan][0] = pos_host.shape[0]


def nf_accel_host(plan: int, acc_host: torch.Tensor) -> None:
    acc_host = _host_f32(acc_host, "acc_host")
    _rows(plan, acc_host, "acc_host")
    _check(_lib.nf_accel_host(plan, ctypes.c_void_p(acc_host.data_ptr())))


def nf_workspace_bytes(plan: int, n: int) -> int:
    return int(_lib.nf_workspace_bytes(plan, int(n)))


def nf_set_workspace(plan: int, ws: torch.Tensor | None) -> None:
    if ws is None:
        _check(_lib.nf_set_workspace(plan, None, 0))
    else:
        _check(_lib.nf_set_workspace(plan, ctypes.c_void_p(ws.data_ptr()), ws.numel() * ws.element_size()))


def nf_set_option(plan: int, key: str, value: int) -> None:
    _check(_lib.nf_set_option(plan, key.encode(), int(value)))


def nf_slab_histogram(plan: int, pos: torch.Tensor, cpd: int) -> list[int]:
    pos = _dev_f32(pos, "pos")
    h = (ctypes.c_longlong * cpd)()
    _check(_lib.nf_slab_histogram(plan, ctypes.c_void_p(pos.data_ptr()), pos.shape[0], h))
    return list(h)


def nf_slab_histogram_static(plan: int, pos: torch.Tensor, cpd: int) -> list[int]:
    """nf_slab_histogram without any allocation on the device side: scratch in a static device array of the library
    (cpd <= 1024; calls that overlap on one GPU race -- include/nf.h)."""
    pos = _dev_f32(pos, "pos")
    h = (ctypes.c_longlong * cpd)()
    _check(_lib.nf_slab_histogram_static(plan, ctypes.c_void_p(pos.data_ptr()), pos.shape[0], h))
    return list(h)


def nf_slab_select(plan: int, pos: torch.Tensor, x_first: int, n_slabs: int, cap: int, want_index: bool = False):
    """Returns (selected positions [m][3], input indices [m] int64 or None); ``cap`` = an upper bound of m."""
    pos = _dev_f32(pos, "pos")
    out = torch.empty((max(int(cap), 0), 3), dtype=torch.float32, device=pos.device)
    idx = torch.empty((max(int(cap), 0),), dtype=torch.int32, device=pos.device) if want_index else None
    m = ctypes.c_longlong(0)
    _check(_lib.nf_slab_select(plan, ctypes.c_void_p(pos.data_ptr()), pos.shape[0], int(x_first), int(n_slabs),
                               ctypes.c_void_p(out.data_ptr()) if out.numel() else None,
                               ctypes.c_void_p(idx.data_ptr()) if (idx is not None and idx.numel()) else None, out.shape[0], ctypes.byref(m)))
    return out[:m.value], (idx[:m.value].to(torch.int64) if idx is not None else None)


def nf_get_slab_cost(plan: int, cpd: int) -> list[float]:
    c = (ctypes.c_double * cpd)()
    _check(_lib.nf_get_slab_cost(plan, c))
    return list(c)


def nf_slab_partition(cost, cpd: int, world: int) -> list[tuple[int, int]]:
    """Host-only: contiguous slab ranges (first, count) with balanced cost; ``cost`` None = equal costs."""
    first, count = (ctypes.c_int * world)(), (ctypes.c_int * world)()
    carr = None
    if cost is not None:
        if len(cost) != cpd:
            raise ValueError("cost must have cpd entries")
        carr = (ctypes.c_double * cpd)(*[float(v) for v in cost])
    _check(_lib.nf_slab_partition(carr, int(cpd), int(world), first, count))
    return [(first[r], count[r]) for r in range(world)]


def nf_get_stats(plan: int) -> dict:
    st = nf_stats()
    _check(_lib.nf_get_stats(plan, ctypes.byref(st)))
    return {name: getattr(st, name) for name, _ in nf_stats._fields_}


class _DevView:
    """Borrowed device memory exposed through __cuda_array_interface__ (copied out by the caller)."""

    def __init__(self, ptr: int, n: int, typestr: str):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": typestr, "data": (ptr, False), "version": 2}


def _copy_out(ptr, n: int, typestr: str, dtype) -> torch.Tensor:
    if n == 0 or not ptr:
        return torch.empty(0, dtype=dtype, device="cuda")
    return torch.as_tensor(_DevView(ptr, n, typestr), device="cuda").clone()


def nf_get_binning(plan: int, n: int, ncells: int) -> dict:
    """Copies of cell_id [n], count [C], offset [C+1], perm [n] as int32-typed CUDA tensors holding the
    uint32 bit patterns (view them as uint32 on the host)."""
    p = [ctypes.c_void_p() for _ in range(4)]
    _check(_lib.nf_get_binning(plan, *[ctypes.byref(q) for q in p]))
    torch.cuda.current_stream().synchronize()
    sizes = [n, ncells, ncells + 1, n]
    names = ["cid", "count", "offset", "perm"]
    return {k: _copy_out(q.value, s, "<i4", torch.int32) for k, q, s in zip(names, p, sizes)}


def nf_get_layout(plan: int, ncells: int) -> dict:
    p = [ctypes.c_void_p() for _ in range(4)]
    sc = ctypes.c_double()
    _check(_lib.nf_get_layout(plan, *[ctypes.byref(q) for q in p], ctypes.byref(sc)))
    poff = _copy_out(p[0].value, ncells + 1, "<i4", torch.int32)
    total = int(poff[-1].item()) & 0xFFFFFFFF
    out = {"poff": poff, "scale": sc.value}
    for k, q in zip("xyz", p[1:]):
        out[k] = _copy_out(q.value, total, "<f4", torch.float32)
    return out


# ---- convenience wrapper ----------------------------------------------------------------------
class Plan:
    """``with Plan(cpd, L, eps, R) as p: p.bin(pos); acc = p.accel()``"""

    def __init__(self, cpd: int, L: float, eps: float, R: int = 2):
        self._h = None
        self.cpd, self.L, self.eps, self.R = int(cpd), float(L), float(eps), int(R)
        self.ncells = self.cpd ** 3
        self.n = 0
        self._h = nf_plan_create(cpd, L, eps, R)

    def close(self):
        if self._h:
            nf_destroy(self._h)
            self._h = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _use_current_stream(self):
        nf_set_stream(self._h, torch.cuda.current_stream().cuda_stream)

    def set_option(self, key: str, value: int):
        nf_set_option(self._h, key, value)

    def set_sink_slabs(self, x_first: int, n_slabs: int):
        nf_set_sink_slabs(self._h, x_first, n_slabs)

    def bin(self, pos: torch.Tensor):
        self._use_current_stream()
        nf_bin(self._h, pos)
        self.n = pos.shape[0]

    def rebin(self, pos: torch.Tensor):
        """Incremental re-binning of the same particles at new positions (same order, same n)."""
        self._use_current_stream()
        nf_rebin(self._h, pos)

    def set_masses(self, mass: torch.Tensor | None):
        """Source masses [n] (input order) of the particles last binned; None = unit masses.  nf_bin resets them."""
        self._use_current_stream()
        nf_set_masses(self._h, mass, self.n)

    def accel(self, out: torch.Tensor | None = None) -> torch.Tensor:
        self._use_current_stream()
        if out is None:
            out = torch.empty((self.n, 3), dtype=torch.float32, device="cuda")
        nf_accel(self._h, out)
        return out

    def accel_density(self, b: float, out: torch.Tensor | None = None, rho: torch.Tensor | None = None):
        """Accelerations and the kernel density estimate of radius ``b`` in one pass; returns (acc, rho)."""
        self._use_current_stream()
        if out is None:
            out = torch.empty((self.n, 3), dtype=torch.float32, device="cuda")
        if rho is None:
            rho = torch.empty((self.n,), dtype=torch.float32, device="cuda")
        nf_accel_density(self._h, out, rho, b)
        return out, rho

    def accel_kick(self, vel: torch.Tensor | None, dt: float, out: torch.Tensor | None = None, want_amax: bool = True,
                   store_acc: bool = True):
        """Accelerations, kick of ``vel`` in place and per-cell max |a| in one pass; returns (acc, amax_cell)."""
        self._use_current_stream()
        if out is None and store_acc:
            out = torch.empty((self.n, 3), dtype=torch.float32, device="cuda")
        if vel is not None and vel.shape[0] != self.n:
            raise ValueError("vel must have one row per binned particle")
        amax = torch.empty((self.ncells,), dtype=torch.float32, device="cuda") if want_amax else None
        nf_accel_kick(self._h, out if store_acc else None, vel, dt, amax)
        return out, amax

    def bin_host(self, pos_host: torch.Tensor):
        self._use_current_stream()
        nf_bin_host(self._h, pos_host)
        self.n = pos_host.shape[0]

    def accel_host(self, out_host: torch.Tensor) -> torch.Tensor:
        self._use_current_stream()
        nf_accel_host(self._h, out_host)
        return out_host

    def slab_histogram(self, pos: torch.Tensor) -> list[int]:
        self._use_current_stream()
        return nf_slab_histogram(self._h, pos, self.cpd)

    def slab_select(self, pos: torch.Tensor, x_first: int, n_slabs: int, cap: int, want_index: bool = False):
        self._use_current_stream()
        return nf_slab_select(self._h, pos, x_first, n_slabs, cap, want_index)

    def slab_cost(self) -> list[float]:
        return nf_get_slab_cost(self._h, self.cpd)

    def binning(self) -> dict:
        return nf_get_binning(self._h, self.n, self.ncells)

    def layout(self) -> dict:
        return nf_get_layout(self._h, self.ncells)

    def stats(self) -> dict:
        return nf_get_stats(self._h)

    def workspace_bytes(self, n: int) -> int:
        return nf_workspace_bytes(self._h, n)

    def set_workspace(self, ws: torch.Tensor | None):
        self._ws = ws
        nf_set_workspace(self._h, ws)
