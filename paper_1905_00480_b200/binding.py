"""Thin ctypes binding over libsho.so (include/sho.h) -- argument marshalling only.

Every step of the hot path runs inside the CUDA kernels of the library; this module validates tensor
shapes / dtypes, passes raw pointers and the CUDA stream handle, and turns status codes into
exceptions.  PyTorch supplies device memory and streams, nothing else.  There is NO CPU fallback: if
libsho.so cannot be loaded (or built) every entry point raises ``ShoError``.
"""
from __future__ import annotations

import ctypes as C
import os
import re

import numpy as np

from . import build as _build

SHO_OK, SHO_ERR_INVALID_ARG, SHO_ERR_UNSUPPORTED, SHO_ERR_OOM, SHO_ERR_CUDA = range(5)
DTYPE_CODES = {"r64": 0, "c128": 1, "r32": 2, "c64": 3}
_NP_OF = {"r64": np.float64, "c128": np.complex128, "r32": np.float32, "c64": np.complex64}


class ShoError(RuntimeError):
    def __init__(self, status, detail, where):
        self.status = int(status)
        super().__init__("%s failed: status %d (%s): %s" % (where, status, _status_name(status), detail))


def _status_name(s):
    return ["SHO_OK", "SHO_ERR_INVALID_ARG", "SHO_ERR_UNSUPPORTED", "SHO_ERR_OOM", "SHO_ERR_CUDA"][s] if 0 <= s < 5 else "?"


def _declared_symbols():
    """Function names declared in include/sho.h (used by the ABI test and to set up ctypes)."""
    with open(os.path.join(_build.INCLUDE, "sho.h")) as f:
        text = f.read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sho_[a-z0-9_]+)\s*\(", text)))


DECLARED_SYMBOLS = _declared_symbols()

_lib = None
_i32p, _i64p, _f64p, _vp = C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.POINTER(C.c_double), C.c_void_p


def lib_path() -> str:
    return _build.LIB


def build_library(force: bool = False) -> str:
    return _build.build_library(force=force)


def lib():
    """Load libsho.so (building it in-tree first if it is missing / stale and nvcc is available)."""
    global _lib
    if _lib is not None:
        return _lib
    try:
        path = _build.build_library()
    except Exception as e:  # no nvcc, or the compile failed
        if os.path.exists(_build.LIB) and "nvcc was not found" in str(e):
            path = _build.LIB   # stale timestamps on a box without nvcc: use what was shipped
        else:
            raise ShoError(SHO_ERR_CUDA, str(e), "loading libsho.so") from e
    try:
        L = C.CDLL(path)
    except OSError as e:
        raise ShoError(SHO_ERR_CUDA, str(e), "loading libsho.so") from e
    L.sho_nsho.argtypes = [C.c_int]; L.sho_nsho.restype = C.c_int
    L.sho_index.argtypes = [C.c_int] * 4; L.sho_index.restype = C.c_int
    L.sho_status_string.argtypes = [C.c_int]; L.sho_status_string.restype = C.c_char_p
    L.sho_last_error.argtypes = []; L.sho_last_error.restype = C.c_char_p
    L.sho_plan_create.argtypes = [C.POINTER(_vp), _i32p, C.c_double, _i32p, _f64p, C.c_int32, _f64p, _f64p,
                                  C.c_int32, C.c_double, C.c_int]
    L.sho_plan_destroy.argtypes = [_vp]
    L.sho_plan_set_option.argtypes = [_vp, C.c_char_p, C.c_int64]
    L.sho_plan_boxes.argtypes = [_vp, _i32p]
    L.sho_plan_info.argtypes = [_vp, _i64p]
    L.sho_project.argtypes = [_vp, _vp, C.c_int32, _vp, _vp]
    L.sho_add.argtypes = [_vp, _vp, C.c_int32, _vp, _vp]
    L.sho_tables_build.argtypes = [_vp, C.POINTER(_vp), C.POINTER(C.c_size_t), _vp]
    L.sho_tables_destroy.argtypes = [_vp]
    L.sho_project_stored.argtypes = [_vp, _vp, _vp, C.c_int32, _vp, _vp]
    L.sho_project_host.argtypes = [_vp, _vp, C.c_int32, _vp, _vp]
    L.sho_add_host.argtypes = [_vp, _vp, C.c_int32, _vp, _vp]
    L.sho_measure_fp64_peak.argtypes = [C.c_int32, _f64p]
    L.sho_rlm_index.argtypes = [C.c_int] * 4; L.sho_rlm_index.restype = C.c_int
    L.sho_umatrix.argtypes = [C.c_int, _f64p]
    L.sho_transform.argtypes = [_vp, _vp, _vp, C.c_int32, _vp, _vp]
    L.sho_add_stored.argtypes = [_vp, _vp, _vp, C.c_int32, _vp, _vp]
    L.sho_tables1d_build.argtypes = [_vp, C.POINTER(_vp), C.POINTER(C.c_size_t), _vp]
    L.sho_tables1d_destroy.argtypes = [_vp]
    L.sho_project_stored1d.argtypes = [_vp, _vp, _vp, C.c_int32, _vp, _vp]
    L.sho_add_stored1d.argtypes = [_vp, _vp, _vp, C.c_int32, _vp, _vp]
    L.sho_project_bf.argtypes = [_vp, _vp, C.c_int32, _vp, _vp, C.c_size_t, _vp]
    L.sho_add_bf.argtypes = [_vp, _vp, C.c_int32, _vp, _vp, C.c_size_t, _vp]
    L.sho_project_bf_static.argtypes = [_vp, _vp, C.c_int32, _vp, _vp]
    L.sho_dmul.argtypes = [_vp, _vp, _vp, C.c_int32, _vp, _vp]
    L.sho_apply.argtypes = [_vp, _vp, _vp, C.c_int32, _vp, _vp]
    L.sho_apply_host.argtypes = [_vp, _vp, _vp, C.c_int32, _vp]
    for name in DECLARED_SYMBOLS:
        fn = getattr(L, name)   # AttributeError here = header and library disagree
        if name not in ("sho_status_string", "sho_last_error", "sho_nsho", "sho_index", "sho_rlm_index"):
            fn.restype = C.c_int
    _lib = L
    return L


def _check(status, where):
    if status != SHO_OK:
        raise ShoError(status, lib().sho_last_error().decode(errors="replace"), where)


def nsho(numax: int) -> int:
    return int(lib().sho_nsho(int(numax)))


def index(nx: int, ny: int, nz: int, numax: int) -> int:
    return int(lib().sho_index(int(nx), int(ny), int(nz), int(numax)))


def rlm_index(nr: int, l: int, m: int, numax: int) -> int:
    return int(lib().sho_rlm_index(int(nr), int(l), int(m), int(numax)))


def umatrix(numax: int) -> np.ndarray:
    """U[rlm_index][index] between Cartesian and spherical SHO states (sho_umatrix; host computation)."""
    n = nsho(numax)
    if n < 0:
        raise ValueError("numax out of range")
    out = np.zeros((n, n), dtype=np.float64)
    _check(lib().sho_umatrix(int(numax), out.ctypes.data_as(_f64p)), "sho_umatrix")
    return out


def _torch():
    import torch
    return torch


def _torch_dtype(dt):
    torch = _torch()
    return {"r64": torch.float64, "c128": torch.complex128, "r32": torch.float32, "c64": torch.complex64}[dt]


def _stream_handle(stream):
    if stream is None:
        return _torch().cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


class Tables:
    """Pre-sampled 3D projector tables (the stored-projector baseline); owned by the library."""

    def __init__(self, plan, handle, nbytes):
        self.plan, self._h, self.nbytes = plan, handle, int(nbytes)

    def close(self):
        if self._h:
            lib().sho_tables_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Tables1D(Tables):
    """Pre-sampled 1D factor tables (the stored-1D separable variant); owned by the library."""

    def close(self):
        if self._h:
            lib().sho_tables1d_destroy(self._h)
            self._h = None


class Plan:
    """Geometry of one set of atoms on one grid (sho_plan_create).  Layouts as in include/sho.h:
    psi [nbands][Nz][Ny][Nx], coeff [natoms][nbands][N_SHO]."""

    def __init__(self, ng, h, periodic, pos, sigma, numax, dtype="r64", kfrac=None, rcut_sigma=6.0):
        L = lib()
        self.ng = tuple(int(x) for x in ng)
        self.h, self.numax, self.dtype, self.rcut_sigma = float(h), int(numax), dtype, float(rcut_sigma)
        if dtype not in DTYPE_CODES:
            raise ValueError("dtype must be one of %s" % list(DTYPE_CODES))
        ng_ = np.ascontiguousarray(ng, dtype=np.int32)
        per_ = np.ascontiguousarray(periodic, dtype=np.int32)
        pos_ = np.ascontiguousarray(pos, dtype=np.float64).reshape(-1, 3)
        sig_ = np.ascontiguousarray(sigma, dtype=np.float64).reshape(-1)
        if pos_.shape[0] != sig_.shape[0]:
            raise ValueError("pos and sigma disagree on the number of atoms")
        kf_ = None if kfrac is None else np.ascontiguousarray(kfrac, dtype=np.float64)
        self.natoms = int(pos_.shape[0])
        self.nsho = nsho(numax)
        h_ = _vp()
        st = L.sho_plan_create(C.byref(h_), ng_.ctypes.data_as(_i32p), float(h), per_.ctypes.data_as(_i32p),
                               None if kf_ is None else kf_.ctypes.data_as(_f64p), self.natoms,
                               pos_.ctypes.data_as(_f64p), sig_.ctypes.data_as(_f64p), int(numax),
                               float(rcut_sigma), DTYPE_CODES[dtype])
        self._h = None
        _check(st, "sho_plan_create")
        self._h = h_
        self.device = _torch().cuda.current_device()      # the plan belongs to the device that was current (sho.h)

    # -- housekeeping ---------------------------------------------------------------------------
    def close(self):
        if self._h:
            lib().sho_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    @property
    def is_complex(self):
        return self.dtype in ("c128", "c64")

    def boxes(self) -> np.ndarray:
        """Integer box ranges [natoms][3][2] = (i_lo, i_hi) per axis, unwrapped (test hook)."""
        out = np.zeros((self.natoms, 3, 2), dtype=np.int32)
        if self.natoms:
            _check(lib().sho_plan_boxes(self._h, out.ctypes.data_as(_i32p)), "sho_plan_boxes")
        return out

    def info(self) -> dict:
        v = np.zeros(8, dtype=np.int64)
        _check(lib().sho_plan_info(self._h, v.ctypes.data_as(_i64p)), "sho_plan_info")
        keys = ("natoms", "nsho", "numax", "dtype", "sum_box_points", "add_tiles", "add_pairs", "atoms_nonempty")
        return dict(zip(keys, (int(x) for x in v)))

    # -- argument checks (marshalling only) -----------------------------------------------------
    def _check_psi(self, psi, where):
        torch = _torch()
        if not (isinstance(psi, torch.Tensor) and psi.is_cuda and psi.is_contiguous()):
            raise ValueError("%s: psi must be a contiguous CUDA tensor" % where)
        if psi.device.index != self.device:
            raise ValueError("%s: psi lives on cuda:%s, the plan on cuda:%d" % (where, psi.device.index, self.device))
        if psi.dtype != _torch_dtype(self.dtype):
            raise ValueError("%s: psi dtype %s does not match the plan (%s)" % (where, psi.dtype, self.dtype))
        if psi.dim() != 4 or tuple(psi.shape[1:]) != (self.ng[2], self.ng[1], self.ng[0]):
            raise ValueError("%s: psi must be [nbands][Nz][Ny][Nx]" % where)
        return int(psi.shape[0])

    def _check_coeff(self, coeff, nb, where):
        torch = _torch()
        if not (isinstance(coeff, torch.Tensor) and coeff.is_cuda and coeff.is_contiguous()):
            raise ValueError("%s: coeff must be a contiguous CUDA tensor" % where)
        if coeff.device.index != self.device:
            raise ValueError("%s: coeff lives on cuda:%s, the plan on cuda:%d" % (where, coeff.device.index, self.device))
        if coeff.dtype != _torch_dtype(self.dtype) or tuple(coeff.shape) != (self.natoms, nb, self.nsho):
            raise ValueError("%s: coeff must be [natoms][nbands][N_SHO] of the plan's dtype" % where)

    def new_coeff(self, nbands, device=None):
        torch = _torch()
        return torch.empty((self.natoms, int(nbands), self.nsho), dtype=_torch_dtype(self.dtype),
                           device=device or torch.device("cuda", torch.cuda.current_device()))

    def set_option(self, key: str, value: int):
        """Tuning / test knob of this plan (include/sho.h: "project_bands_per_cta", "host_chunk_bands"; 0 = automatic)."""
        _check(lib().sho_plan_set_option(self._h, key.encode(), int(value)), "sho_plan_set_option")
        return self

    # -- the hot calls ---------------------------------------------------------------------------
    def project(self, psi, coeff=None, stream=None):
        nb = self._check_psi(psi, "sho_project")
        if coeff is None:
            coeff = self.new_coeff(nb, psi.device)
        self._check_coeff(coeff, nb, "sho_project")
        _check(lib().sho_project(self._h, psi.data_ptr(), nb, coeff.data_ptr(), _stream_handle(stream)), "sho_project")
        return coeff

    def add(self, coeff, psi, stream=None):
        nb = self._check_psi(psi, "sho_add")
        self._check_coeff(coeff, nb, "sho_add")
        _check(lib().sho_add(self._h, coeff.data_ptr(), nb, psi.data_ptr(), _stream_handle(stream)), "sho_add")
        return psi

    def _check_dmat(self, dmat, where):
        torch = _torch()
        if not (isinstance(dmat, torch.Tensor) and dmat.is_cuda and dmat.is_contiguous() and dmat.dtype == torch.float64
                and tuple(dmat.shape) == (self.natoms, self.nsho, self.nsho) and dmat.device.index == self.device):
            raise ValueError("%s: dmat must be a contiguous float64 CUDA tensor [natoms][N_SHO][N_SHO] on the plan's device" % where)

    def dmul(self, dmat, coeff, out=None, stream=None):
        """Step (2): out[a][b][i] = sum_j dmat[a][i][j] coeff[a][b][j] (out may be coeff itself)."""
        nb = int(coeff.shape[1])
        self._check_coeff(coeff, nb, "sho_dmul")
        self._check_dmat(dmat, "sho_dmul")
        if out is None:
            out = self.new_coeff(nb, coeff.device)
        self._check_coeff(out, nb, "sho_dmul")
        _check(lib().sho_dmul(self._h, dmat.data_ptr(), coeff.data_ptr(), nb, out.data_ptr(), _stream_handle(stream)), "sho_dmul")
        return out

    def transform(self, umat, coeff, out=None, stream=None):
        """out[a][b][i] = sum_j umat[i][j] coeff[a][b][j]: one [N_SHO][N_SHO] matrix for all atoms (sho_transform)."""
        torch = _torch()
        nb = int(coeff.shape[1])
        self._check_coeff(coeff, nb, "sho_transform")
        if not (isinstance(umat, torch.Tensor) and umat.is_cuda and umat.is_contiguous() and umat.dtype == torch.float64
                and tuple(umat.shape) == (self.nsho, self.nsho) and umat.device.index == self.device):
            raise ValueError("sho_transform: umat must be a contiguous float64 CUDA tensor [N_SHO][N_SHO] on the plan's device")
        if out is None:
            out = self.new_coeff(nb, coeff.device)
        self._check_coeff(out, nb, "sho_transform")
        _check(lib().sho_transform(self._h, umat.data_ptr(), coeff.data_ptr(), nb, out.data_ptr(), _stream_handle(stream)), "sho_transform")
        return out

    def apply(self, dmat, psi, coeff_work=None, stream=None):
        """psi += add(dmat * project(psi)): the three steps of the non-local action on one stream."""
        nb = self._check_psi(psi, "sho_apply")
        self._check_dmat(dmat, "sho_apply")
        if coeff_work is None:
            coeff_work = self.new_coeff(nb, psi.device)
        self._check_coeff(coeff_work, nb, "sho_apply")
        _check(lib().sho_apply(self._h, dmat.data_ptr(), psi.data_ptr(), nb, coeff_work.data_ptr(), _stream_handle(stream)),
               "sho_apply")
        return psi

    # -- band-fastest psi [Nz][Ny][Nx][nbands] (the paper's layout) ------------------------------
    def _check_psi_bf(self, psi, where):
        torch = _torch()
        if not (isinstance(psi, torch.Tensor) and psi.is_cuda and psi.is_contiguous() and psi.device.index == self.device):
            raise ValueError("%s: psi_bf must be a contiguous CUDA tensor on the plan's device" % where)
        if psi.dtype != _torch_dtype(self.dtype) or psi.dim() != 4 or tuple(psi.shape[:3]) != (self.ng[2], self.ng[1], self.ng[0]):
            raise ValueError("%s: psi_bf must be [Nz][Ny][Nx][nbands] of the plan's dtype" % where)
        return int(psi.shape[3])

    def _work(self, work, nb, where):
        torch = _torch()
        if work is None:                 # convenience: a workspace of at most 64 bands
            n = min(nb, 64)
            work = torch.empty((n, self.ng[2], self.ng[1], self.ng[0]), dtype=_torch_dtype(self.dtype),
                               device=torch.device("cuda", self.device))
        if not (isinstance(work, torch.Tensor) and work.is_cuda and work.is_contiguous() and work.device.index == self.device):
            raise ValueError("%s: work must be a contiguous CUDA tensor on the plan's device" % where)
        return work

    def project_bf(self, psi_bf, coeff=None, work=None, stream=None):
        nb = self._check_psi_bf(psi_bf, "sho_project_bf")
        if coeff is None:
            coeff = self.new_coeff(nb, psi_bf.device)
        self._check_coeff(coeff, nb, "sho_project_bf")
        work = self._work(work, nb, "sho_project_bf")
        _check(lib().sho_project_bf(self._h, psi_bf.data_ptr(), nb, coeff.data_ptr(), work.data_ptr(),
                                    work.numel() * work.element_size(), _stream_handle(stream)), "sho_project_bf")
        return coeff

    def project_bf_static(self, psi_bf, coeff=None, stream=None):
        """sho_project_bf without a workspace argument: the library converts the band chunks in its own fixed
        32 MiB device array (STATIC_WORK_BYTES), so the C call allocates nothing.  Meant for callers that own only
        psi_bf and coeff (see include/sho.h); pass ``coeff`` to keep this wrapper from allocating the output too.
        Calls on one device share that array: keep them on one stream.  ShoError (SHO_ERR_UNSUPPORTED) if one band
        of the grid is larger than the array."""
        nb = self._check_psi_bf(psi_bf, "sho_project_bf_static")
        if coeff is None:
            coeff = self.new_coeff(nb, psi_bf.device)
        self._check_coeff(coeff, nb, "sho_project_bf_static")
        _check(lib().sho_project_bf_static(self._h, psi_bf.data_ptr(), nb, coeff.data_ptr(), _stream_handle(stream)),
               "sho_project_bf_static")
        return coeff

    def add_bf(self, coeff, psi_bf, work=None, stream=None):
        nb = self._check_psi_bf(psi_bf, "sho_add_bf")
        self._check_coeff(coeff, nb, "sho_add_bf")
        work = self._work(work, nb, "sho_add_bf")
        _check(lib().sho_add_bf(self._h, coeff.data_ptr(), nb, psi_bf.data_ptr(), work.data_ptr(),
                                work.numel() * work.element_size(), _stream_handle(stream)), "sho_add_bf")
        return psi_bf

    def tables_bytes(self) -> int:
        need = C.c_size_t(0)
        _check(lib().sho_tables_build(self._h, None, C.byref(need), None), "sho_tables_build(size query)")
        return int(need.value)

    def tables(self, stream=None) -> Tables:
        need = C.c_size_t(0)
        h_ = _vp()
        st = lib().sho_tables_build(self._h, C.byref(h_), C.byref(need), _stream_handle(stream))
        _check(st, "sho_tables_build")
        return Tables(self, h_, need.value)

    def project_stored(self, tables, psi, coeff=None, stream=None):
        nb = self._check_psi(psi, "sho_project_stored")
        if coeff is None:
            coeff = self.new_coeff(nb, psi.device)
        self._check_coeff(coeff, nb, "sho_project_stored")
        _check(lib().sho_project_stored(self._h, tables._h, psi.data_ptr(), nb, coeff.data_ptr(),
                                        _stream_handle(stream)), "sho_project_stored")
        return coeff

    def add_stored(self, tables, coeff, psi, stream=None):
        nb = self._check_psi(psi, "sho_add_stored")
        self._check_coeff(coeff, nb, "sho_add_stored")
        _check(lib().sho_add_stored(self._h, tables._h, coeff.data_ptr(), nb, psi.data_ptr(), _stream_handle(stream)), "sho_add_stored")
        return psi

    def tables1d_bytes(self) -> int:
        need = C.c_size_t(0)
        _check(lib().sho_tables1d_build(self._h, None, C.byref(need), None), "sho_tables1d_build(size query)")
        return int(need.value)

    def tables1d(self, stream=None) -> Tables1D:
        need = C.c_size_t(0)
        h_ = _vp()
        _check(lib().sho_tables1d_build(self._h, C.byref(h_), C.byref(need), _stream_handle(stream)), "sho_tables1d_build")
        return Tables1D(self, h_, need.value)

    def project_stored1d(self, tables, psi, coeff=None, stream=None):
        nb = self._check_psi(psi, "sho_project_stored1d")
        if coeff is None:
            coeff = self.new_coeff(nb, psi.device)
        self._check_coeff(coeff, nb, "sho_project_stored1d")
        _check(lib().sho_project_stored1d(self._h, tables._h, psi.data_ptr(), nb, coeff.data_ptr(), _stream_handle(stream)),
               "sho_project_stored1d")
        return coeff

    def add_stored1d(self, tables, coeff, psi, stream=None):
        nb = self._check_psi(psi, "sho_add_stored1d")
        self._check_coeff(coeff, nb, "sho_add_stored1d")
        _check(lib().sho_add_stored1d(self._h, tables._h, coeff.data_ptr(), nb, psi.data_ptr(), _stream_handle(stream)),
               "sho_add_stored1d")
        return psi

    # -- end-to-end with HOST buffers (numpy arrays or pinned CPU tensors) ------------------------
    def _host_ptr(self, a, shape, where):
        torch = _torch()
        if isinstance(a, torch.Tensor):
            if a.is_cuda or not a.is_contiguous() or a.dtype != _torch_dtype(self.dtype) or tuple(a.shape) != shape:
                raise ValueError("%s: host tensor has the wrong device / layout / dtype / shape" % where)
            return a.data_ptr()
        if not (isinstance(a, np.ndarray) and a.flags.c_contiguous and a.dtype == _NP_OF[self.dtype] and a.shape == shape):
            raise ValueError("%s: host array has the wrong layout / dtype / shape" % where)
        return a.ctypes.data

    def project_host(self, psi_host, coeff_host, stream=None):
        nb = int(psi_host.shape[0])
        pp = self._host_ptr(psi_host, (nb, self.ng[2], self.ng[1], self.ng[0]), "sho_project_host")
        cp = self._host_ptr(coeff_host, (self.natoms, nb, self.nsho), "sho_project_host")
        _check(lib().sho_project_host(self._h, pp, nb, cp, _stream_handle(stream)), "sho_project_host")
        return coeff_host

    def apply_host(self, dmat_host, psi_host, stream=None):
        nb = int(psi_host.shape[0])
        pp = self._host_ptr(psi_host, (nb, self.ng[2], self.ng[1], self.ng[0]), "sho_apply_host")
        torch = _torch()
        shape = (self.natoms, self.nsho, self.nsho)
        if isinstance(dmat_host, torch.Tensor):
            if dmat_host.is_cuda or not dmat_host.is_contiguous() or dmat_host.dtype != torch.float64 or tuple(dmat_host.shape) != shape:
                raise ValueError("sho_apply_host: dmat must be a contiguous float64 host tensor [natoms][N_SHO][N_SHO]")
            dp = dmat_host.data_ptr()
        else:
            if not (isinstance(dmat_host, np.ndarray) and dmat_host.flags.c_contiguous and dmat_host.dtype == np.float64
                    and dmat_host.shape == shape):
                raise ValueError("sho_apply_host: dmat must be a C-contiguous float64 array [natoms][N_SHO][N_SHO]")
            dp = dmat_host.ctypes.data
        _check(lib().sho_apply_host(self._h, dp, pp, nb, _stream_handle(stream)), "sho_apply_host")
        return psi_host

    def add_host(self, coeff_host, psi_host, stream=None):
        nb = int(psi_host.shape[0])
        pp = self._host_ptr(psi_host, (nb, self.ng[2], self.ng[1], self.ng[0]), "sho_add_host")
        cp = self._host_ptr(coeff_host, (self.natoms, nb, self.nsho), "sho_add_host")
        _check(lib().sho_add_host(self._h, cp, nb, pp, _stream_handle(stream)), "sho_add_host")
        return psi_host


# same names as the C ABI, for callers that prefer functions
def sho_project(plan: Plan, psi, coeff=None, stream=None):
    return plan.project(psi, coeff, stream)


def sho_add(plan: Plan, coeff, psi, stream=None):
    return plan.add(coeff, psi, stream)


def sho_project_stored(plan: Plan, tables: Tables, psi, coeff=None, stream=None):
    return plan.project_stored(tables, psi, coeff, stream)


def sho_add_stored(plan: Plan, tables: Tables, coeff, psi, stream=None):
    return plan.add_stored(tables, coeff, psi, stream)


def sho_project_stored1d(plan: Plan, tables: Tables1D, psi, coeff=None, stream=None):
    return plan.project_stored1d(tables, psi, coeff, stream)


def sho_add_stored1d(plan: Plan, tables: Tables1D, coeff, psi, stream=None):
    return plan.add_stored1d(tables, coeff, psi, stream)


def sho_project_bf(plan: Plan, psi_bf, coeff=None, work=None, stream=None):
    return plan.project_bf(psi_bf, coeff, work, stream)


def sho_add_bf(plan: Plan, coeff, psi_bf, work=None, stream=None):
    return plan.add_bf(coeff, psi_bf, work, stream)


STATIC_WORK_BYTES = 32 << 20        # SHO_STATIC_WORK_BYTES of include/sho.h


def sho_project_bf_static(plan: Plan, psi_bf, coeff=None, stream=None):
    return plan.project_bf_static(psi_bf, coeff, stream)


def sho_transform(plan: Plan, umat, coeff, out=None, stream=None):
    return plan.transform(umat, coeff, out, stream)


def sho_dmul(plan: Plan, dmat, coeff, out=None, stream=None):
    return plan.dmul(dmat, coeff, out, stream)


def sho_apply(plan: Plan, dmat, psi, coeff_work=None, stream=None):
    return plan.apply(dmat, psi, coeff_work, stream)


def sho_apply_host(plan: Plan, dmat_host, psi_host, stream=None):
    return plan.apply_host(dmat_host, psi_host, stream)


def sho_project_host(plan: Plan, psi_host, coeff_host, stream=None):
    return plan.project_host(psi_host, coeff_host, stream)


def sho_add_host(plan: Plan, coeff_host, psi_host, stream=None):
    return plan.add_host(coeff_host, psi_host, stream)


def measure_fp64_peak(iters: int = 20000) -> float:
    """Achieved FLOP/s of a DFMA-chain micro-kernel on every SM (roofline denominator for bench.py)."""
    out = C.c_double(0.0)
    _check(lib().sho_measure_fp64_peak(int(iters), C.byref(out)), "sho_measure_fp64_peak")
    return float(out.value)


def plan_for(w, dtype=None) -> Plan:
    """Plan for a ``workloads.Workload``."""
    return Plan(w.ng, w.h, w.periodic, w.pos, w.sigma, w.numax, dtype or w.dtype, w.kfrac, w.rcut_sigma)
