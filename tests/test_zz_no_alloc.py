"""sho_project_bf_static: the band-fastest projection for callers that cannot allocate device memory.

Why the entry point exists.  ``sho_project_bf`` wants a device workspace from its caller.  Some users of this
library have none to give: a plug-in that runs inside a DFT program which reserved the whole GPU for its own
memory arena at start-up (a cudaMalloc made later simply fails), or a routine called while that program's other
streams are busy (cudaMalloc / cudaFree synchronise the device and would stall them).  They are handed psi and
coeff and own nothing else.  ``sho_project_bf_static`` converts the band chunks in a fixed 32 MiB device array
that is part of libsho.so itself, so the call allocates nothing; the price is a size limit (one band of the grid
must fit in 32 MiB) and that all calls on a device share the one array.

What is checked here: the new entry point against the existing ``sho_project_bf`` path (which the parity tests
compare with the oracle), in the norm and at the tolerance of tests/test_gpu_parity.py (reading A13: max |dc| /
||psi_b|| <= 1e-12 for fp64), on TWO calls in a row.  The second call has other data and fewer bands than the
first, so anything it wrongly picked up from what the first call left in the shared array would show.  The grid
is the paper's own 64^3, where 16 fp64 bands fit in the array: 40 bands make three chunks, the last
one short.  The size limit must be reported as an error, not overrun.

This file is named so that pytest collects it last: a failure here must not hide the parity tests under ``-x``.
It needs nothing from the other test files and passes alone in a fresh process as well as after them (the first
call on a device is the one that looks up the array's address; either order of tests makes it here or earlier).
"""
import numpy as np
import pytest

from paper_1905_00480_b200 import workloads

pytestmark = pytest.mark.gpu

TOL = 1e-12          # fp64, same as tests/test_gpu_parity.py


@pytest.fixture(scope="module")
def sho():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    import paper_1905_00480_b200 as pkg
    pkg.lib()          # raises if libsho.so cannot be loaded: no silent fallback
    return pkg


def _psi_bf(w, nb, first_band):
    """Seeded psi_bf[Nz][Ny][Nx][nb] on the device and the per-band norms ||psi_b|| = sqrt(h^3 sum |psi|^2)."""
    import torch
    psi = w.psi(range(first_band, first_band + nb))                     # [nb][Nz][Ny][Nx]
    norm = np.sqrt(w.h ** 3 * np.sum(np.abs(psi.astype(np.float64)) ** 2, axis=(1, 2, 3)))
    return torch.from_numpy(np.ascontiguousarray(np.moveaxis(psi, 0, 3))).cuda(), norm


def _compare(got, ref, norm):
    got, ref = got.cpu().numpy(), ref.cpu().numpy()
    assert np.all(np.isfinite(got))
    assert np.abs(ref).max() > 0.0                                       # the reference path did project something
    err = (np.abs(got - ref) / norm[None, :, None]).max()
    assert err <= TOL, "static-workspace projection differs from sho_project_bf: %.3e > %.1e" % (err, TOL)


def test_static_workspace_projection_matches_the_workspace_path_on_two_calls_in_a_row(sho):
    import torch
    w = workloads.make_paper(5, "r64", size="full")                      # 64^3 isolated, 665 atoms, numax 5
    band_bytes = w.npoints * 8
    assert sho.STATIC_WORK_BYTES // band_bytes == 16                     # so 40 bands are chunks of 16, 16, 8
    plan = sho.plan_for(w)
    try:
        for nb, first_band in ((40, 0), (5, 100)):                       # call 1, then call 2 with other data, fewer bands
            psi_bf, norm = _psi_bf(w, nb, first_band)
            # the existing path, with a caller workspace of 6 bands (so its chunks differ from the static path's)
            work = torch.empty((6, w.ng[2], w.ng[1], w.ng[0]), dtype=psi_bf.dtype, device="cuda")
            ref = plan.project_bf(psi_bf, work=work)
            # the new path; its output buffer is poisoned first so that every element must have been written
            out = torch.full_like(ref, float("nan"))
            got = plan.project_bf_static(psi_bf, coeff=out)
            torch.cuda.synchronize()
            assert got.data_ptr() == out.data_ptr()
            _compare(got, ref, norm)
    finally:
        plan.close()


def test_static_workspace_rejects_a_grid_whose_band_does_not_fit(sho):
    import torch
    ng = (256, 256, 65)                                                  # 34.1 MB per fp64 band > 32 MiB
    assert ng[0] * ng[1] * ng[2] * 8 > sho.STATIC_WORK_BYTES
    pos = np.array([[6.0, 6.0, 6.0]])
    plan = sho.Plan(ng, 0.25, (1, 1, 1), pos, np.array([0.5]), 2, "r64")
    try:
        psi_bf = torch.zeros((ng[2], ng[1], ng[0], 1), dtype=torch.float64, device="cuda")
        coeff = torch.full((1, 1, plan.nsho), 7.0, dtype=torch.float64, device="cuda")
        with pytest.raises(sho.ShoError) as ei:
            plan.project_bf_static(psi_bf, coeff=coeff)
        assert ei.value.status == 2                                      # SHO_ERR_UNSUPPORTED
        assert "SHO_STATIC_WORK_BYTES" in str(ei.value)
        torch.cuda.synchronize()
        assert bool((coeff == 7.0).all())                                # nothing was launched
        # the same grid goes through the path that takes the caller's workspace
        work = torch.empty((1, ng[2], ng[1], ng[0]), dtype=torch.float64, device="cuda")
        plan.project_bf(psi_bf, coeff=coeff, work=work)
        torch.cuda.synchronize()
        assert bool((coeff == 0.0).all())                                # psi is zero
    finally:
        plan.close()
