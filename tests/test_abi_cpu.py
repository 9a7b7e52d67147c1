"""CPU-side checks of libsho.so: it builds, loads, exports every symbol include/sho.h declares, its
integer host functions agree with the paper / the oracle, and without a GPU it fails LOUDLY (no CPU
fallback).  No compute call is made here."""
import ctypes
import os
import re
import subprocess

import numpy as np
import pytest

import oracle
import paper_1905_00480_b200 as sho
from paper_1905_00480_b200 import build as sho_build
from paper_1905_00480_b200 import workloads

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_and_exports_every_declared_symbol():
    path = sho.build_library()
    assert os.path.exists(path)
    L = ctypes.CDLL(path)
    assert len(sho.DECLARED_SYMBOLS) >= 16
    for name in ("sho_project", "sho_add", "sho_project_stored"):      # the calls north_star names
        assert name in sho.DECLARED_SYMBOLS
    for name in sho.DECLARED_SYMBOLS:
        assert hasattr(L, name), "include/sho.h declares %s but libsho.so does not export it" % name
    out = subprocess.run(["nm", "-D", "--defined-only", path], capture_output=True, text=True).stdout
    exported = set(re.findall(r" T (sho_\w+)", out))
    assert exported == set(sho.DECLARED_SYMBOLS), "exported C symbols and the header disagree"


def test_header_has_no_torch_or_cxx_types():
    with open(os.path.join(ROOT, "include", "sho.h")) as f:
        text = f.read()
    assert 'extern "C"' in text
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)      # declarations only (comments may mention torch layouts)
    for bad in ("torch", "at::", "std::", "Tensor", "template"):
        assert bad not in text


def test_kernels_are_compiled_for_sm_100a_with_fp64_tensor_core_mma():
    path = sho.build_library()
    r = subprocess.run(["cuobjdump", "-lelf", path], capture_output=True, text=True)
    assert "sm_100a" in r.stdout
    assert "-lineinfo" in sho_build.NVCC_FLAGS and "arch=compute_100a,code=sm_100a" in sho_build.NVCC_FLAGS


def test_nsho_matches_paper_values(golden):
    for numax, n in golden("nsho_paper.txt"):
        assert sho.nsho(int(numax)) == int(n)
    assert sho.nsho(7) == 120 and sho.nsho(9) == 220 and sho.nsho(15) == 816
    assert sho.nsho(-1) == -1 and sho.nsho(16) == -1


def test_index_map_is_the_oracles_enumeration():
    for numax in range(0, 16):
        seen = []
        for nz in range(numax + 1):
            for ny in range(numax + 1 - nz):
                for nx in range(numax + 1 - nz - ny):
                    i = sho.index(nx, ny, nz, numax)
                    assert i == oracle.index(nx, ny, nz, numax)
                    seen.append(i)
        assert seen == list(range(sho.nsho(numax)))           # nx fastest, then ny, then nz (reading A8)
        assert sho.index(numax + 1, 0, 0, numax) == -1 and sho.index(0, -1, 0, numax) == -1


def test_status_strings():
    L = sho.lib()
    assert L.sho_status_string(0) == b"SHO_OK"
    assert L.sho_status_string(2) == b"SHO_ERR_UNSUPPORTED"


def _no_gpu():
    import torch
    return not torch.cuda.is_available()


def test_invalid_arguments_are_rejected_before_any_cuda_call():
    w = workloads.make(1)
    bad = [
        dict(h=-0.25), dict(h=float("nan")), dict(numax=-1), dict(numax=16), dict(rcut_sigma=0.0),
        dict(sigma=[-1.0]), dict(ng=(32, 0, 32)), dict(kfrac=(0.1, 0.0, 0.0)),       # kfrac needs a complex dtype
        dict(pos=[[float("inf"), 0, 0]]),
    ]
    for kw in bad:
        a = dict(ng=w.ng, h=w.h, periodic=w.periodic, pos=w.pos, sigma=w.sigma, numax=w.numax, rcut_sigma=6.0, kfrac=None)
        a.update(kw)
        with pytest.raises(sho.ShoError) as ei:
            sho.Plan(a["ng"], a["h"], a["periodic"], a["pos"], a["sigma"], a["numax"], "r64", a["kfrac"], a["rcut_sigma"])
        assert ei.value.status == 1, kw
    with pytest.raises(sho.ShoError) as ei:     # periodic box wider than the cell: valid problem, not covered on the GPU
        sho.Plan((16, 16, 16), 0.25, (1, 1, 1), [[1.0, 1.0, 1.0]], [1.0], 2)
    assert ei.value.status == 2


@pytest.mark.skipif(not _no_gpu(), reason="checks the behaviour WITHOUT a CUDA device")
def test_no_cpu_fallback_without_a_device():
    w = workloads.make(1)
    with pytest.raises(sho.ShoError) as ei:
        sho.plan_for(w)
    assert ei.value.status == 4                       # SHO_ERR_CUDA: the product path fails loudly
    with pytest.raises(sho.ShoError):
        sho.measure_fp64_peak(10)


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1905_00480_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                with open(os.path.join(dirpath, fn)) as f:
                    text = f.read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), fn
                assert "sho_oracle" not in text, fn
    with open(os.path.join(ROOT, "oracle", "sho_oracle.c")) as f:
        otext = f.read()
    assert "#include \"sho" not in otext and "paper_1905_00480_b200/" not in otext.replace("(paper_1905_00480_b200/csrc)", "")


def test_workload_generator_is_seeded_and_shaped_like_the_configs():
    for k, (ng, na, nb, numax, dt) in {1: ((32,) * 3, 1, 1, 3, "r64"), 2: ((96,) * 3, 32, 16, 5, "r64"),
                                        3: ((128,) * 3, 256, 32, 7, "r64"), 4: ((128,) * 3, 512, 32, 7, "r64"),
                                        5: ((192,) * 3, 1024, 64, 9, "c128")}.items():
        w = workloads.make(k)
        assert (w.ng, w.natoms, w.nbands, w.numax, w.dtype) == (ng, na, nb, numax, dt)
        w2 = workloads.make(k)
        assert np.array_equal(w.pos, w2.pos) and np.array_equal(w.sigma, w2.sigma)
    w = workloads.make(2, size="small")
    assert np.array_equal(w.psi_band(1), w.psi()[1])
    assert not np.array_equal(w.psi_band(0), w.psi_band(1))


def test_umatrix_and_rlm_index_match_the_oracle():
    """sho_umatrix is host code (no GPU): the library's exact quadrature against the oracle's, and the spherical
    index map against the oracle's literal enumeration."""
    for numax in (0, 1, 2, 4, 7, 9):
        U = sho.umatrix(numax)
        Uo = oracle.umatrix(numax)
        assert U.shape == Uo.shape and np.max(np.abs(U - Uo)) < 1e-13
        for nu in range(numax + 1):
            for nr in range(nu // 2 + 1):
                l = nu - 2 * nr
                for m in range(-l, l + 1):
                    assert sho.rlm_index(nr, l, m, numax) == oracle.rlm_index(nr, l, m, numax)
    assert sho.rlm_index(0, 3, 0, 2) == -1 and sho.rlm_index(0, 1, 2, 3) == -1
