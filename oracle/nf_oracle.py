"""ctypes binding of ``nf_oracle.c`` (argument marshalling only; the arithmetic is in C).

TEST INFRASTRUCTURE ONLY -- see the package docstring.  PAPER.md:337-349 (sec. 3.1) is
the passage the C file follows.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nf_oracle.c")
_LIB = os.path.join(_HERE, "libnf_oracle.so")
_lib = None


class OracleError(RuntimeError):
    pass


def build(force: bool = False) -> str:
    """Compile ``nf_oracle.c`` with gcc -O2 (no fast-math) + OpenMP.  Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i64, f64, i32 = ctypes.c_int64, ctypes.c_double, ctypes.c_int
        vp = ctypes.c_void_p
        lib.nfo_num_threads.restype = i32
        lib.nfo_kernel.restype = f64
        lib.nfo_kernel.argtypes = [f64, f64]
        lib.nfo_bin.restype = i32
        lib.nfo_bin.argtypes = [vp, i64, i32, f64, vp, vp, vp, vp]
        lib.nfo_kernel_plummer.restype = f64
        lib.nfo_kernel_plummer.argtypes = [f64, f64]
        lib.nfo_accel_kind.restype = i32
        lib.nfo_accel_kind.argtypes = [vp, i64, i32, f64, f64, i32, i32, vp, vp, vp, vp, i64, vp]
        lib.nfo_accel_mass.restype = i32
        lib.nfo_accel_mass.argtypes = [vp, vp, i64, i32, f64, f64, i32, i32, vp, vp, vp, vp, i64, vp]
        lib.nfo_accel.restype = i32
        lib.nfo_accel.argtypes = [vp, i64, i32, f64, f64, i32, vp, vp, vp, vp, i64, vp]
        lib.nfo_density.restype = i32
        lib.nfo_density.argtypes = [vp, i64, i32, f64, f64, i32, vp, vp, vp, vp, i64, vp]
        lib.nfo_force_scale.restype = i32
        lib.nfo_force_scale.argtypes = [vp, vp, i64, i32, f64, f64, i32, i32, vp, vp, vp, vp, i64, vp]
        lib.nfo_interactions.restype = i64
        lib.nfo_interactions.argtypes = [vp, i32, i32]
        _lib = lib
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        name = {-1: "ARG", -2: "DOMAIN", -3: "NOMEM"}.get(rc, str(rc))
        raise OracleError(f"{what} failed: NFO_ERR_{name}")


def _pos32(pos) -> np.ndarray:
    pos = np.ascontiguousarray(pos, dtype=np.float32)
    if pos.ndim != 2 or pos.shape[1] != 3:
        raise ValueError("pos must be [n][3]")
    return pos


def num_threads() -> int:
    return int(_load().nfo_num_threads())


def kernel(r: float, eps: float, softening: str = "spline") -> float:
    """K(r): the acceleration on a sink from a unit-mass source at displacement d is d*K(|d|)."""
    if softening == "plummer":
        return float(_load().nfo_kernel_plummer(float(r), float(eps)))
    return float(_load().nfo_kernel(float(r), float(eps)))


def bin_particles(pos, cpd: int, L: float):
    """Returns dict(cid, count, offset, perm) as uint32 arrays."""
    pos = _pos32(pos)
    n = pos.shape[0]
    C = cpd ** 3
    cid = np.empty(n, np.uint32)
    count = np.empty(C, np.uint32)
    offset = np.empty(C + 1, np.uint32)
    perm = np.empty(n, np.uint32)
    rc = _load().nfo_bin(pos.ctypes.data, n, cpd, float(L), cid.ctypes.data, count.ctypes.data,
                         offset.ctypes.data, perm.ctypes.data)
    _check(rc, "nfo_bin")
    return {"cid": cid, "count": count, "offset": offset, "perm": perm}


def accel(pos, cpd: int, L: float, eps: float, R: int = 2, sinks=None, binning=None, softening: str = "spline") -> np.ndarray:
    """float64 accelerations [m][3]; ``sinks`` = input indices to evaluate (default: all, input order).
    ``softening``: "spline" (the method) or "plummer" (the paper's comparison law)."""
    kind = {"spline": 0, "plummer": 1}[softening]
    pos = _pos32(pos)
    n = pos.shape[0]
    if binning is None:
        binning = bin_particles(pos, cpd, L)
    if sinks is None:
        sp, m = None, n
    else:
        sinks = np.ascontiguousarray(sinks, dtype=np.int64)
        sp, m = sinks.ctypes.data, sinks.shape[0]
    acc = np.zeros((m, 3), np.float64)
    rc = _load().nfo_accel_kind(pos.ctypes.data, n, cpd, float(L), float(eps), int(R), kind,
                           binning["cid"].ctypes.data, binning["offset"].ctypes.data,
                           binning["perm"].ctypes.data, sp, m, acc.ctypes.data)
    _check(rc, "nfo_accel")
    return acc


def accel_mass(pos, mass, cpd: int, L: float, eps: float, R: int = 2, sinks=None, binning=None,
               softening: str = "spline") -> np.ndarray:
    """float64 accelerations [m][3] with per-particle source masses: a_i = sum_j m_j d_ij K(r_ij)
    (the direct sum of PAPER.md:349 with the mass written out; ``mass`` float32 [n], input order)."""
    kind = {"spline": 0, "plummer": 1}[softening]
    pos = _pos32(pos)
    n = pos.shape[0]
    mass = np.ascontiguousarray(mass, dtype=np.float32)
    if mass.shape != (n,):
        raise ValueError("mass must have shape (n,)")
    if binning is None:
        binning = bin_particles(pos, cpd, L)
    if sinks is None:
        sp, m = None, n
    else:
        sinks = np.ascontiguousarray(sinks, dtype=np.int64)
        sp, m = sinks.ctypes.data, sinks.shape[0]
    acc = np.zeros((m, 3), np.float64)
    rc = _load().nfo_accel_mass(pos.ctypes.data, mass.ctypes.data, n, cpd, float(L), float(eps), int(R), kind,
                                binning["cid"].ctypes.data, binning["offset"].ctypes.data,
                                binning["perm"].ctypes.data, sp, m, acc.ctypes.data)
    _check(rc, "nfo_accel_mass")
    return acc


def density(pos, cpd: int, L: float, b: float, R: int = 2, sinks=None, binning=None) -> np.ndarray:
    """float64 kernel density estimate [m]: sum over the stencil of max(0, 1 - r^2/b^2), self included."""
    pos = _pos32(pos)
    n = pos.shape[0]
    if binning is None:
        binning = bin_particles(pos, cpd, L)
    if sinks is None:
        sp, m = None, n
    else:
        sinks = np.ascontiguousarray(sinks, dtype=np.int64)
        sp, m = sinks.ctypes.data, sinks.shape[0]
    rho = np.zeros(m, np.float64)
    rc = _load().nfo_density(pos.ctypes.data, n, cpd, float(L), float(b), int(R),
                             binning["cid"].ctypes.data, binning["offset"].ctypes.data,
                             binning["perm"].ctypes.data, sp, m, rho.ctypes.data)
    _check(rc, "nfo_density")
    return rho


def force_scale(pos, cpd: int, L: float, eps: float, R: int = 2, sinks=None, binning=None, softening: str = "spline",
                mass=None) -> np.ndarray:
    """float64 [m]: S_i = sum_j m_j |d_ij| K(|d_ij|) over the stencil of sink i -- the uncancelled magnitude of the
    direct sum (reading C13): the scale a float32 evaluation's error is proportional to."""
    kind = {"spline": 0, "plummer": 1}[softening]
    pos = _pos32(pos)
    n = pos.shape[0]
    mp = None
    if mass is not None:
        mass = np.ascontiguousarray(mass, dtype=np.float32)
        if mass.shape != (n,):
            raise ValueError("mass must have shape (n,)")
        mp = mass.ctypes.data
    if binning is None:
        binning = bin_particles(pos, cpd, L)
    if sinks is None:
        sp, m = None, n
    else:
        sinks = np.ascontiguousarray(sinks, dtype=np.int64)
        sp, m = sinks.ctypes.data, sinks.shape[0]
    out = np.zeros(m, np.float64)
    rc = _load().nfo_force_scale(pos.ctypes.data, mp, n, cpd, float(L), float(eps), int(R), kind,
                                 binning["cid"].ctypes.data, binning["offset"].ctypes.data,
                                 binning["perm"].ctypes.data, sp, m, out.ctypes.data)
    _check(rc, "nfo_force_scale")
    return out


def kick(vel, acc, dt: float) -> np.ndarray:
    """Leapfrog kick v + a dt in float64 ("kicks the particle velocities")."""
    return np.asarray(vel, np.float64) + np.asarray(acc, np.float64) * float(dt)


def cell_max_accel(acc, cid, ncells: int) -> np.ndarray:
    """Per-cell maximum of the Euclidean norm of the particle accelerations, 0 for empty cells: "the per-cell
    maximum particle acceleration" of the timestep criterion.  acc [n][3], cid [n] cell ids."""
    norm = np.sqrt((np.asarray(acc, np.float64) ** 2).sum(axis=1))
    out = np.zeros(int(ncells), np.float64)
    np.maximum.at(out, np.asarray(cid, np.int64), norm)
    return out


def interactions(count, cpd: int, R: int = 2) -> int:
    """Exact ordered-pair count of the definition (self pairs included)."""
    count = np.ascontiguousarray(count, dtype=np.uint32)
    v = int(_load().nfo_interactions(count.ctypes.data, cpd, R))
    if v < 0:
        raise OracleError("nfo_interactions: cpd < 2R+1")
    return v
