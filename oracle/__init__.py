"""CPU oracle for the Landau gauge-fixing hot path -- TEST INFRASTRUCTURE, not the product.

Thin ctypes loader around ``oracle/lgf_oracle.c`` (plain C11, double precision, Algorithm 1 of
arXiv:1206.0675 step by step; see the header of that file for conventions and citations).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It imports nothing from ``paper_1206_0675_b200`` and the CUDA path
imports nothing from here.

Array conventions (numpy, complex128, C-contiguous):
  links U : shape (Lt, Lz, Ly, Lx, 4, 3, 3)   site-major, mu = 0..3 = x, y, z, t
  Delta, w, g : shape (Lt, Lz, Ly, Lx, 3, 3)
  scalar field : shape (Lt, Lz, Ly, Lx)
  dims : (Lx, Ly, Lz, Lt)   (x fastest in memory)
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lgf_oracle.c")
_SRC_HB = os.path.join(_HERE, "lgf_heatbath_oracle.c")      # thermalisation oracle
_LIB = os.path.join(_HERE, "liblgf_oracle.so")
CFLAGS = ["-O2", "-std=c11", "-fopenmp", "-fcx-limited-range", "-shared", "-fPIC"]

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (idempotent).  Returns the path of the shared object."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_HB))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.run(["gcc", *CFLAGS, _SRC, _SRC_HB, "-o", tmp, "-lm"], check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        vp, i4 = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int)
        dp, d, lg = ctypes.POINTER(ctypes.c_double), ctypes.c_double, ctypes.c_long
        lib.orc_num_threads.restype = ctypes.c_int
        lib.orc_measure.argtypes = [i4, vp, vp, dp, dp]
        lib.orc_dft4d.argtypes = [i4, vp, ctypes.c_int, vp]
        lib.orc_p2.argtypes = [i4, i4]
        lib.orc_p2.restype = d
        lib.orc_accelerate.argtypes = [i4, vp, vp]
        lib.orc_build_g.argtypes = [i4, vp, d, vp]
        lib.orc_transform.argtypes = [i4, vp, vp]
        lib.orc_iterate.argtypes = [i4, vp, d, lg, vp, vp]
        lib.orc_fix.argtypes = [i4, vp, d, d, lg, vp, vp, lg]
        lib.orc_fix.restype = lg
        lib.orc_plaquette.argtypes = [i4, vp]
        lib.orc_plaquette.restype = d
        lib.orc_gs.argtypes = [vp, vp]
        lib.orc_reconstruct_row3.argtypes = [vp, vp]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().orc_num_threads())


def _dims(dims):
    dims = tuple(int(v) for v in dims)
    assert len(dims) == 4
    return dims, (ctypes.c_int * 4)(*dims)


def _c128(a, shape):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    assert a.shape == tuple(shape), (a.shape, shape)
    return a


def _site_shape(dims):
    return (dims[3], dims[2], dims[1], dims[0])


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def measure(dims, U, want_delta: bool = True):
    """Alg. 1 line 1 / 17.  Returns (Delta or None, F, theta)."""
    dims, cd = _dims(dims)
    U = _c128(U, _site_shape(dims) + (4, 3, 3))
    Delta = np.empty(_site_shape(dims) + (3, 3), np.complex128) if want_delta else None
    F, th = ctypes.c_double(), ctypes.c_double()
    _load().orc_measure(cd, _ptr(U), _ptr(Delta) if want_delta else None, ctypes.byref(F), ctypes.byref(th))
    return Delta, F.value, th.value


def dft4d(dims, f, sign: int):
    """Naive separable 4-D DFT of one complex scalar field; sign=-1 forward, +1 inverse, unnormalised."""
    dims, cd = _dims(dims)
    f = _c128(f, _site_shape(dims))
    out = np.empty_like(f)
    _load().orc_dft4d(cd, _ptr(f), int(sign), _ptr(out))
    return out


def gluon_field(dims, U, mu: int):
    """A_mu(k) = sum_x exp(-2 pi i k.x/L) A_mu(x), unnormalised: shape (Lt, Lz, Ly, Lx, 3, 3) indexed by (kt, kz, ky, kx)."""
    dims, cd = _dims(dims)
    U = _c128(U, _site_shape(dims) + (4, 3, 3))
    Ak = np.empty(_site_shape(dims) + (3, 3), np.complex128)
    _load().orc_gluon_field(cd, _ptr(U), int(mu), _ptr(Ak))
    return Ak


def p2(dims, k):
    dims, cd = _dims(dims)
    return float(_load().orc_p2(cd, (ctypes.c_int * 4)(*[int(v) for v in k])))


def accelerate(dims, Delta):
    """Alg. 1 lines 3-8: w = F^-1 (16/p^2) F Delta, zero mode removed, 1/V included."""
    dims, cd = _dims(dims)
    Delta = _c128(Delta, _site_shape(dims) + (3, 3))
    w = np.empty_like(Delta)
    _load().orc_accelerate(cd, _ptr(Delta), _ptr(w))
    return w


def build_g(dims, w, alpha: float):
    dims, cd = _dims(dims)
    w = _c128(w, _site_shape(dims) + (3, 3))
    g = np.empty_like(w)
    _load().orc_build_g(cd, _ptr(w), float(alpha), _ptr(g))
    return g


def transform(dims, U, g):
    """Returns g(x) U_mu(x) g(x+mu)^dag as a new array."""
    dims, cd = _dims(dims)
    U = _c128(U, _site_shape(dims) + (4, 3, 3)).copy()
    g = _c128(g, _site_shape(dims) + (3, 3))
    _load().orc_transform(cd, _ptr(U), _ptr(g))
    return U


def iterate(dims, U, alpha: float, n: int):
    """n updates.  Returns (U_after, F[0..n], theta[0..n]); entry i = after i updates (R12)."""
    dims, cd = _dims(dims)
    U = _c128(U, _site_shape(dims) + (4, 3, 3)).copy()
    Fh = np.zeros(n + 1)
    Th = np.zeros(n + 1)
    _load().orc_iterate(cd, _ptr(U), float(alpha), int(n), _ptr(Fh), _ptr(Th))
    return U, Fh, Th


def fix(dims, U, alpha: float, tol: float, max_iter: int):
    """Algorithm 1.  Returns (U_fixed, iterations, F[0..it], theta[0..it])."""
    dims, cd = _dims(dims)
    U = _c128(U, _site_shape(dims) + (4, 3, 3)).copy()
    cap = int(max_iter) + 1
    Fh = np.zeros(cap)
    Th = np.zeros(cap)
    it = int(_load().orc_fix(cd, _ptr(U), float(alpha), float(tol), int(max_iter), _ptr(Fh), _ptr(Th), cap))
    return U, it, Fh[: it + 1].copy(), Th[: it + 1].copy()


def plaquette(dims, U) -> float:
    dims, cd = _dims(dims)
    U = _c128(U, _site_shape(dims) + (4, 3, 3))
    return float(_load().orc_plaquette(cd, _ptr(U)))


def gs(M):
    """Gram-Schmidt projection of one 3x3 complex matrix onto SU(3) (rows; R9)."""
    M = _c128(M, (3, 3))
    G = np.empty_like(M)
    _load().orc_gs(_ptr(M), _ptr(G))
    return G


def reconstruct_row3(rows01):
    rows01 = _c128(rows01, (2, 3))
    out = np.empty(3, np.complex128)
    _load().orc_reconstruct_row3(_ptr(rows01), _ptr(out))
    return out


# ---- thermalisation oracle (lgf_heatbath_oracle.c) -------------------------
def hb_staples(dims, U):
    """Staple sums A_mu(x) of every link: shape (Lt, Lz, Ly, Lx, 4, 3, 3); Re tr[U A] sums the plaquettes
    that contain the link."""
    dims, cd = _dims(dims)
    U = _c128(U, _site_shape(dims) + (4, 3, 3))
    A = np.empty_like(U)
    _load().orc_hb_staples(cd, _ptr(U), _ptr(A))
    return A


def hb_kp_sample(a: float, seed: int, n: int):
    """n Kennedy-Pendleton draws X ~ exp(a x0) sqrt(1 - x0^2) dx0 dOmega.  Returns (X[n, 4], attempts[n])."""
    X = np.empty((n, 4), np.float64)
    att = np.empty(n, np.int32)
    lib = _load()
    lib.orc_hb_kp_sample.argtypes = [ctypes.c_double, ctypes.c_ulonglong, ctypes.c_long, ctypes.c_void_p, ctypes.c_void_p]
    lib.orc_hb_kp_sample(float(a), int(seed), int(n), X.ctypes.data, att.ctypes.data)
    return X, att


def heatbath(dims, U, beta: float, seed: int, sweep0: int, nsweeps: int):
    """nsweeps Cabibbo-Marinari heat-bath sweeps (numbered from sweep0) of the Wilson action at beta.
    Returns the new configuration."""
    dims, cd = _dims(dims)
    U = _c128(U, _site_shape(dims) + (4, 3, 3)).copy()
    lib = _load()
    lib.orc_heatbath.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_double, ctypes.c_ulonglong, ctypes.c_long,
                                 ctypes.c_long]
    lib.orc_heatbath.restype = ctypes.c_int
    rc = lib.orc_heatbath(cd, _ptr(U), float(beta), int(seed), int(sweep0), int(nsweeps))
    if rc != 0:
        raise ValueError("heatbath needs even lattice extents")
    return U


def overrelax(dims, U, nsweeps: int):
    """nsweeps microcanonical overrelaxation sweeps (R28): the action is conserved.  Returns the new configuration."""
    dims, cd = _dims(dims)
    U = _c128(U, _site_shape(dims) + (4, 3, 3)).copy()
    lib = _load()
    lib.orc_overrelax.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_long]
    lib.orc_overrelax.restype = ctypes.c_int
    if lib.orc_overrelax(cd, _ptr(U), int(nsweeps)) != 0:
        raise ValueError("overrelax needs even lattice extents")
    return U
