"""ctypes wrapper around oracle/sho_oracle.c (argument marshalling only; no arithmetic here).

TEST INFRASTRUCTURE, NOT THE PRODUCT: see the header of sho_oracle.c.  ``build()`` compiles the C
file with gcc (-O2 -fopenmp -ffp-contract=off) into oracle/libsho_oracle.so.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sho_oracle.c")
_LIB = os.path.join(_HERE, "libsho_oracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle if the .so is missing or older than the source."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + ".tmp.%d" % os.getpid()
            cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
                   "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, _LIB)
    return _LIB


_i32p = C.POINTER(C.c_int32)
_f64p = C.POINTER(C.c_double)


def _load():
    global _lib
    if _lib is None:
        build()
        lib = C.CDLL(_LIB)
        lib.oracle_num_threads.restype = C.c_int
        lib.oracle_nsho.argtypes = [C.c_int]
        lib.oracle_index.argtypes = [C.c_int] * 4
        lib.oracle_hermite_phys.argtypes = [C.c_int, C.c_double]
        lib.oracle_hermite_phys.restype = C.c_double
        lib.oracle_phi.argtypes = [C.c_int, C.c_double, C.c_double]
        lib.oracle_phi.restype = C.c_double
        lib.oracle_box.argtypes = [_i32p, C.c_double, _i32p, _f64p, C.c_double, C.c_double, _i32p, _i32p]
        common = [_i32p, C.c_double, _i32p, _f64p, C.c_int, _f64p, _f64p, C.c_int, C.c_double, C.c_int, C.c_int]
        lib.oracle_project.argtypes = common + [_f64p, _f64p]
        lib.oracle_project_pairs.argtypes = common + [_f64p, C.POINTER(_f64p), C.c_int64, _i32p, _i32p, _f64p]
        lib.oracle_add.argtypes = common + [_f64p, _f64p]
        lib.oracle_add_points.argtypes = common + [_f64p, C.c_int64, _i32p, _i32p, _f64p]
        lib.oracle_dmul.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, _f64p, _f64p, _f64p]
        lib.oracle_add_points_bands.argtypes = common + [_f64p, C.c_int64, _i32p, C.c_int, _i32p, _f64p]
        _lib = lib
    return _lib


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a, t):
    return a.ctypes.data_as(t)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def nsho(numax: int) -> int:
    return int(_load().oracle_nsho(int(numax)))


def index(nx: int, ny: int, nz: int, numax: int) -> int:
    return int(_load().oracle_index(int(nx), int(ny), int(nz), int(numax)))


def hermite_phys(n: int, xi: float) -> float:
    return float(_load().oracle_hermite_phys(int(n), float(xi)))


def phi(n: int, u: float, sigma: float) -> float:
    return float(_load().oracle_phi(int(n), float(u), float(sigma)))


def box(ng, h, periodic, pos, sigma, rcut_sigma=6.0):
    """(lo[3], hi[3], empty) of one atom; reading A3/A5."""
    ng_, per_, pos_ = _i32(ng), _i32(periodic), _f64(pos)
    lo = np.zeros(3, np.int32)
    hi = np.zeros(3, np.int32)
    e = _load().oracle_box(_p(ng_, _i32p), float(h), _p(per_, _i32p), _p(pos_, _f64p), float(sigma),
                           float(rcut_sigma), _p(lo, _i32p), _p(hi, _i32p))
    return lo, hi, bool(e)


def _common(ng, h, periodic, kfrac, pos, sigma, numax, rcut_sigma, is_complex, nbands):
    ng_, per_ = _i32(ng), _i32(periodic)
    pos_ = _f64(pos).reshape(-1, 3)
    sig_ = _f64(sigma).reshape(-1)
    assert pos_.shape[0] == sig_.shape[0]
    kf_ = None if kfrac is None else _f64(kfrac)
    keep = (ng_, per_, pos_, sig_, kf_)
    args = [_p(ng_, _i32p), float(h), _p(per_, _i32p), None if kf_ is None else _p(kf_, _f64p),
            int(pos_.shape[0]), _p(pos_, _f64p), _p(sig_, _f64p), int(numax), float(rcut_sigma),
            int(bool(is_complex)), int(nbands)]
    return args, keep


def _as_real_view(a, is_complex):
    """psi / coeff as a contiguous float64 array (complex128 viewed as interleaved re,im)."""
    a = np.ascontiguousarray(a, dtype=np.complex128 if is_complex else np.float64)
    return a, (a.view(np.float64) if is_complex else a)


def project(ng, h, periodic, kfrac, pos, sigma, numax, psi, rcut_sigma=6.0):
    """coeff[natoms][nbands][N_SHO]; psi [nbands][Nz][Ny][Nx], float64 or complex128."""
    is_complex = np.iscomplexobj(psi)
    psi_, psi_r = _as_real_view(psi, is_complex)
    nb = psi_.shape[0]
    assert psi_.shape[1:] == (ng[2], ng[1], ng[0]), "psi must be [nb][Nz][Ny][Nx]"
    args, keep = _common(ng, h, periodic, kfrac, pos, sigma, numax, rcut_sigma, is_complex, nb)
    na = args[4]
    out = np.zeros((na, nb, nsho(numax)), dtype=np.complex128 if is_complex else np.float64)
    rc = _load().oracle_project(*args, _p(psi_r, _f64p), _p(out.view(np.float64), _f64p))
    assert rc == 0, "oracle_project failed"
    del keep
    return out


def project_pairs(ng, h, periodic, kfrac, pos, sigma, numax, psi_bands, pair_atom, pair_band, nbands,
                  is_complex, rcut_sigma=6.0):
    """Projection of selected (atom, band) pairs.  ``psi_bands`` maps band index -> array [Nz][Ny][Nx]
    (only the bands that occur in ``pair_band`` need to be present)."""
    pa, pb = _i32(pair_atom), _i32(pair_band)
    args, keep = _common(ng, h, periodic, kfrac, pos, sigma, numax, rcut_sigma, is_complex, nbands)
    ptrs = (_f64p * int(nbands))()
    hold = {}
    for b, arr in psi_bands.items():
        a_, r_ = _as_real_view(arr, is_complex)
        assert a_.shape == (ng[2], ng[1], ng[0])
        hold[b] = (a_, r_)
        ptrs[int(b)] = _p(r_, _f64p)
    for b in np.unique(pb):
        assert int(b) in hold, "band %d missing from psi_bands" % b
    out = np.zeros((len(pa), nsho(numax)), dtype=np.complex128 if is_complex else np.float64)
    rc = _load().oracle_project_pairs(*args, None, ptrs, len(pa), _p(pa, _i32p), _p(pb, _i32p),
                                      _p(out.view(np.float64), _f64p))
    assert rc == 0, "oracle_project_pairs failed"
    del keep, hold
    return out


def add(ng, h, periodic, kfrac, pos, sigma, numax, coeff, psi, rcut_sigma=6.0):
    """Returns psi + A c (a new array); coeff [natoms][nbands][N_SHO]."""
    is_complex = np.iscomplexobj(psi) or np.iscomplexobj(coeff)
    psi_, psi_r = _as_real_view(np.array(psi, copy=True), is_complex)
    c_, c_r = _as_real_view(coeff, is_complex)
    nb = psi_.shape[0]
    assert psi_.shape[1:] == (ng[2], ng[1], ng[0])
    args, keep = _common(ng, h, periodic, kfrac, pos, sigma, numax, rcut_sigma, is_complex, nb)
    assert c_.shape == (args[4], nb, nsho(numax))
    rc = _load().oracle_add(*args, _p(c_r, _f64p), _p(psi_r, _f64p))
    assert rc == 0, "oracle_add failed"
    del keep
    return psi_


def add_points(ng, h, periodic, kfrac, pos, sigma, numax, coeff, pts, bands, rcut_sigma=6.0):
    """(A c)(r_j) -- the increment only -- at sample points pts[ns][3] = (jx,jy,jz), band bands[ns]."""
    is_complex = np.iscomplexobj(coeff)
    c_, c_r = _as_real_view(coeff, is_complex)
    nb = c_.shape[1]
    args, keep = _common(ng, h, periodic, kfrac, pos, sigma, numax, rcut_sigma, is_complex, nb)
    pts_, b_ = _i32(pts).reshape(-1, 3), _i32(bands).reshape(-1)
    assert len(pts_) == len(b_)
    out = np.zeros(len(b_), dtype=np.complex128 if is_complex else np.float64)
    rc = _load().oracle_add_points(*args, _p(c_r, _f64p), len(b_), _p(pts_, _i32p), _p(b_, _i32p),
                                   _p(out.view(np.float64), _f64p))
    assert rc == 0, "oracle_add_points failed"
    del keep
    return out


def add_points_bands(ng, h, periodic, kfrac, pos, sigma, numax, coeff, pts, band_sel, rcut_sigma=6.0):
    """(A c)(r_j) -- the increment only -- at sample points pts[ns][3] = (jx,jy,jz) for every band in
    ``band_sel``: out[ns][len(band_sel)]."""
    is_complex = np.iscomplexobj(coeff)
    c_, c_r = _as_real_view(coeff, is_complex)
    nb = c_.shape[1]
    args, keep = _common(ng, h, periodic, kfrac, pos, sigma, numax, rcut_sigma, is_complex, nb)
    pts_, b_ = _i32(pts).reshape(-1, 3), _i32(band_sel).reshape(-1)
    out = np.zeros((len(pts_), len(b_)), dtype=np.complex128 if is_complex else np.float64)
    rc = _load().oracle_add_points_bands(*args, _p(c_r, _f64p), len(pts_), _p(pts_, _i32p), len(b_), _p(b_, _i32p),
                                         _p(out.view(np.float64), _f64p))
    assert rc == 0, "oracle_add_points_bands failed"
    del keep
    return out


def dmul(D, coeff):
    """Step (2): d[a][b][i] = sum_j D[a][i][j] c[a][b][j]; D real [natoms][n][n]."""
    is_complex = np.iscomplexobj(coeff)
    c_, c_r = _as_real_view(coeff, is_complex)
    D_ = _f64(D)
    na, nb, n = c_.shape
    assert D_.shape == (na, n, n)
    out = np.zeros_like(c_)
    rc = _load().oracle_dmul(na, nb, n, int(is_complex), _p(D_, _f64p), _p(c_r, _f64p),
                             _p(out.view(np.float64) if is_complex else out, _f64p))
    assert rc == 0, "oracle_dmul failed"
    return out
