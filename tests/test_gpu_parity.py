"""GPU parity: the CUDA path (through the C ABI of libsho.so) against the CPU oracle, element by element,
on the same seeded inputs (paper_1905_00480_b200.workloads).  Run with ``-m gpu`` on a B200.

Tolerances (north_star / reading A13):
  project: max_b max_{a,n} |c_gpu - c_ref| / ||psi_b||      <= 1e-12 (fp64), 1e-5 (fp32),
           ||psi_b|| = sqrt(h^3 sum_r |psi_b(r)|^2)
  add:     max_b max_r |psi_gpu - psi_ref| / max_r |psi_ref,b| <= 1e-12 (fp64), 1e-5 (fp32)
Integer work (box ranges, index map) must agree exactly.
"""
import numpy as np
import pytest

import oracle
from paper_1905_00480_b200 import workloads

pytestmark = pytest.mark.gpu

TOL = {"r64": 1e-12, "c128": 1e-12, "r32": 1e-5, "c64": 1e-5}
NP_OF = {"r64": np.float64, "c128": np.complex128, "r32": np.float32, "c64": np.complex64}


@pytest.fixture(scope="module")
def sho():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    import paper_1905_00480_b200 as pkg
    pkg.lib()          # raises if libsho.so cannot be loaded: no silent fallback
    return pkg


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _psi_norm(psi, h):
    return np.sqrt(h ** 3 * np.sum(np.abs(psi.astype(np.complex128 if np.iscomplexobj(psi) else np.float64)) ** 2,
                                   axis=(1, 2, 3)))


def _oracle_boxes(w):
    out = np.zeros((w.natoms, 3, 2), np.int32)
    for a in range(w.natoms):
        lo, hi, _ = oracle.box(w.ng, w.h, w.periodic, w.pos[a], w.sigma[a], w.rcut_sigma)
        out[a, :, 0], out[a, :, 1] = lo, hi
    return out


def check_project(sho, w, psi, coeff_gpu, tol, pairs=None):
    """Compare coeff_gpu [na][nb][nsho] (numpy) with the oracle (all pairs, or the listed (a,b) pairs)."""
    wide = np.complex128 if w.is_complex else np.float64
    norm = _psi_norm(psi, w.h)
    if pairs is None:
        ref = oracle.project(w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax, psi.astype(wide), w.rcut_sigma)
        err = np.abs(coeff_gpu.astype(wide) - ref) / np.maximum(norm, 1e-300)[None, :, None]
    else:
        pa, pb = np.array([p[0] for p in pairs]), np.array([p[1] for p in pairs])
        bands = {int(b): psi[int(b)].astype(wide) for b in np.unique(pb)}
        ref = oracle.project_pairs(w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax, bands, pa, pb,
                                   psi.shape[0], w.is_complex, w.rcut_sigma)
        err = np.abs(coeff_gpu[pa, pb].astype(wide) - ref) / norm[pb][:, None]
    assert np.all(np.isfinite(coeff_gpu))
    assert err.max() <= tol, "project parity: max normalised error %.3e > %.1e" % (err.max(), tol)
    return float(err.max())


def run_case(sho, w, stored=True, tol=None, options=None):
    """boxes, project, add, stored project of one workload against the oracle (full comparison).  ``options``:
    sho_plan_set_option knobs to set on the plan first."""
    import torch
    tol = tol or TOL[w.dtype]
    wide = np.complex128 if w.is_complex else np.float64
    plan = sho.plan_for(w)
    try:
        for key, value in (options or {}).items():
            plan.set_option(key, value)
        assert np.array_equal(plan.boxes(), _oracle_boxes(w)), "integer box ranges differ from the oracle"
        assert plan.nsho == oracle.nsho(w.numax)
        psi = w.psi()
        if w.psi_dist == "zero":     # cfg 4 has psi_0 = 0; project needs something to project
            psi = workloads.Workload(**{**w.__dict__, "psi_dist": "normal"}).psi()
        d_psi = _dev(psi)
        # ---- project ----
        c_gpu = plan.project(d_psi)
        torch.cuda.synchronize()
        e_prj = check_project(sho, w, psi, c_gpu.cpu().numpy(), tol)
        # ---- stored-projector baseline ----
        if stored:
            tb = plan.tables()
            c_sto = plan.project_stored(tb, d_psi)
            torch.cuda.synchronize()
            check_project(sho, w, psi, c_sto.cpu().numpy(), tol)
            tb.close()
        # ---- add ----
        coeff = w.coeff(plan.nsho)
        psi0 = w.psi()
        d_psi0 = _dev(psi0)
        plan.add(_dev(coeff), d_psi0)
        torch.cuda.synchronize()
        got = d_psi0.cpu().numpy()
        ref = oracle.add(w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax, coeff.astype(wide), psi0.astype(wide),
                         w.rcut_sigma)
        scale = np.maximum(np.abs(ref).max(axis=(1, 2, 3)), 1e-300)
        err = (np.abs(got.astype(wide) - ref).max(axis=(1, 2, 3)) / scale).max()
        assert err <= tol, "add parity: max normalised error %.3e > %.1e" % (err, tol)
        # ---- f3: the separable kernels on stored 1D tables, and the stored (3D tables) add-back ----
        t1 = plan.tables1d()
        c_1d = plan.project_stored1d(t1, d_psi)
        d_psi1 = _dev(psi0)
        plan.add_stored1d(t1, _dev(coeff), d_psi1)
        torch.cuda.synchronize()
        t1.close()
        check_project(sho, w, psi, c_1d.cpu().numpy(), tol)
        e1 = (np.abs(d_psi1.cpu().numpy().astype(wide) - ref).max(axis=(1, 2, 3)) / scale).max()
        assert e1 <= tol, "stored-1D add parity: %.3e > %.1e" % (e1, tol)
        if stored:
            tb = plan.tables()
            d_psi2 = _dev(psi0)
            plan.add_stored(tb, _dev(coeff), d_psi2)
            torch.cuda.synchronize()
            tb.close()
            e2 = (np.abs(d_psi2.cpu().numpy().astype(wide) - ref).max(axis=(1, 2, 3)) / scale).max()
            assert e2 <= tol, "stored add parity: %.3e > %.1e" % (e2, tol)
        return e_prj, float(err)
    finally:
        plan.close()


# ------------------------------------------------------------------------------------------------
# configs at sizes the oracle finishes in seconds


def test_cfg1_full_single_atom_isolated(sho):
    e = run_case(sho, workloads.make(1))
    assert e[0] < 1e-13 and e[1] < 1e-13        # the contract is loose by orders of magnitude


@pytest.mark.parametrize("dtype", ["r32", "c128", "c64"])
def test_cfg1_other_dtypes(sho, dtype):
    run_case(sho, workloads.make(1, dtype=dtype))


@pytest.mark.parametrize("k", [2, 3, 4, 5])
def test_small_configs_native_dtype(sho, k):
    run_case(sho, workloads.make(k, size="small"))


@pytest.mark.parametrize("k,dtype", [(4, "r32"), (5, "c64"), (2, "c128"), (3, "r32")])
def test_small_configs_other_dtypes(sho, k, dtype):
    w = workloads.make(k, size="small", dtype=dtype)
    if dtype in ("r32", "r64"):
        w.kfrac = None
    run_case(sho, w)


# ------------------------------------------------------------------------------------------------
# edge cases


def _custom(ng, periodic, pos, sigma, numax, nb, dtype="r64", h=0.25, kfrac=None, seed=7, rc=6.0):
    return workloads.Workload("custom", seed, tuple(ng), h, tuple(periodic), kfrac, np.asarray(pos, float).reshape(-1, 3),
                              np.asarray(sigma, float).reshape(-1), numax, nb, dtype, "normal", rcut_sigma=rc)


def test_no_atoms(sho):
    import torch
    w = _custom((16, 16, 16), (1, 1, 1), np.zeros((0, 3)), np.zeros(0), 3, 2)
    plan = sho.plan_for(w)
    psi = _dev(w.psi())
    before = psi.clone()
    c = plan.project(psi)
    assert tuple(c.shape) == (0, 2, 20)
    plan.add(c, psi)
    torch.cuda.synchronize()
    assert torch.equal(psi, before)
    plan.close()


def test_atoms_outside_and_straddling_an_isolated_grid(sho):
    # atom 0 far outside (empty box => exact zeros), atom 1 straddles a corner, atom 2 inside
    pos = [[-30.0, 2.0, 2.0], [0.1, 5.9, 0.3], [3.0, 3.1, 2.9]]
    w = _custom((24, 28, 20), (0, 0, 0), pos, [0.5, 0.45, 0.4], 4, 3)
    import torch
    plan = sho.plan_for(w)
    c = plan.project(_dev(w.psi()))
    torch.cuda.synchronize()
    assert torch.count_nonzero(c[0]) == 0
    plan.close()
    run_case(sho, w)


@pytest.mark.parametrize("periodic", [(1, 1, 1), (1, 0, 1), (0, 1, 0)])
def test_odd_ragged_grid_dims(sho, periodic):
    # Nx odd: the vector loads fall back to scalar; tiles of the add kernel are ragged on every axis
    rng = np.random.default_rng(11)
    ng = (33, 37, 29)
    pos = rng.uniform(0, 1, (5, 3)) * np.array(ng) * 0.25
    run_case(sho, _custom(ng, periodic, pos, rng.uniform(0.35, 0.6, 5), 5, 2))


@pytest.mark.parametrize("numax", [0, 1, 2, 3, 4, 6, 8, 9, 11, 12, 15])
def test_every_numax_tile_shape(sho, numax):
    rng = np.random.default_rng(100 + numax)
    ng = (20, 24, 18)
    pos = rng.uniform(0, 1, (2, 3)) * np.array(ng) * 0.3
    # small sigma and a 4-sigma cut keep the box (9-10 points) inside the cell; parity does not need a wide cut
    run_case(sho, _custom(ng, (1, 1, 1), pos, [0.3, 0.36], numax, 2, h=0.3, rc=4.0), stored=numax <= 9)


@pytest.mark.parametrize("numax", [8, 9])
@pytest.mark.parametrize("dtype", ["r64", "r32", "c128", "c64"])
def test_remainder_rows_every_dtype(sho, numax, dtype):
    # numax 8, 9: the project kernel runs rows ny, nx = 8, 9 as DFMA partials beside the MMA tile.  Boxes of
    # ~29 points wrap on x and y (atom near the origin), span several x chunks and a ragged last y group;
    # complex data carry a Bloch phase on every axis.
    rng = np.random.default_rng(300 + numax)
    ng = (44, 40, 36)
    pos = np.array([[0.4, 0.7, 5.0], [6.1, 5.3, 0.2], [10.2, 9.4, 8.1]])
    kfrac = (0.1, 0.2, 0.3) if dtype in ("c128", "c64") else None
    w = _custom(ng, (1, 1, 1), pos, rng.uniform(0.55, 0.62, 3), numax, 2, dtype=dtype, h=0.25, kfrac=kfrac)
    run_case(sho, w, stored=False)


def test_many_pairs_per_tile_wrap_the_ring(sho):
    # 60 atoms whose boxes all cover the same add tiles: the mbarrier ring of the add kernel (<= 18 pairs)
    # wraps several times, every producer warp reuses its slots and buffers
    rng = np.random.default_rng(5)
    ng = (16, 64, 16)
    pos = (np.array(ng) * 0.25 / 2)[None, :] + rng.uniform(-0.4, 0.4, (60, 3))
    run_case(sho, _custom(ng, (1, 1, 1), pos, rng.uniform(0.3, 0.33, 60), 4, 2, rc=5.0), stored=False)
    run_case(sho, _custom(ng, (1, 1, 1), pos, rng.uniform(0.3, 0.33, 60), 9, 2, dtype="c128", kfrac=(0.1, 0.2, 0.3), rc=5.0),
             stored=False)


@pytest.mark.parametrize("nb", [1, 3])
def test_odd_number_of_real_bands(sho, nb):
    # the add kernel pairs real bands into two channels per CTA: the last CTA has an idle channel
    rng = np.random.default_rng(17)
    ng = (24, 40, 16)
    pos = rng.uniform(0, 1, (6, 3)) * np.array(ng) * 0.25
    run_case(sho, _custom(ng, (1, 1, 1), pos, rng.uniform(0.3, 0.36, 6), 5, nb, rc=4.0), stored=False)
    run_case(sho, _custom(ng, (1, 1, 1), pos, rng.uniform(0.3, 0.36, 6), 5, nb, dtype="r32", rc=4.0), stored=False)


@pytest.mark.parametrize("nx", [18, 22, 36])
def test_bloch_image_boundary_inside_a_load_step(sho, nx):
    # complex128, Nx a multiple of the 2-element lane span but not of the 8-column step: the x-image
    # boundary of a wrapping atom falls inside a step, which the project kernel schedules twice with
    # complementary column masks around the accumulator rotation
    rng = np.random.default_rng(nx)
    ng = (nx, 20, 16)
    L = np.array(ng) * 0.25
    pos = np.stack([np.array([0.3, 2.0, 2.0]), np.array([L[0] - 0.2, 3.0, 1.0]), np.array([L[0] / 2, 0.1, 3.9])])
    run_case(sho, _custom(ng, (1, 1, 1), pos, [0.3, 0.34, 0.32], 9, 2, dtype="c128", kfrac=(0.17, 0.2, 0.3), rc=5.0))
    run_case(sho, _custom(ng, (1, 1, 1), pos, [0.3, 0.34, 0.32], 6, 3, dtype="c64", kfrac=(0.17, -0.2, 0.3), rc=5.0))


def _sample_atoms(w, boxes):
    """Atoms for sampled full-size parity: boxes that wrap on all three axes, the sigma extremes, interior
    boxes (no wrap at all), the first and the last atom -- at least 8 distinct atoms."""
    ng = np.array(w.ng)
    wrap_all = [a for a in range(w.natoms) if all(boxes[a, d, 0] < 0 or boxes[a, d, 1] >= ng[d] for d in range(3))]
    wrap_none = [a for a in range(w.natoms) if all(boxes[a, d, 0] >= 0 and boxes[a, d, 1] < ng[d] for d in range(3))]
    wrap_some = [a for a in range(w.natoms) if a not in wrap_all and a not in wrap_none]
    pick = wrap_all[:3] + wrap_none[:2] + wrap_some[:2] + [int(np.argmin(w.sigma)), int(np.argmax(w.sigma)), 0, w.natoms - 1]
    atoms = []
    for a in pick + list(range(w.natoms)):
        if a not in atoms:
            atoms.append(a)
        if len(atoms) >= 8 and all(x in atoms for x in pick):
            break
    return atoms


def _sample_bands(nb, n=8):
    """First, last and interior bands (the add kernel's work item index runs over bands)."""
    return sorted(set([0, 1, nb // 3, nb // 2 - 1, nb // 2, (2 * nb) // 3 + 1, nb - 2, nb - 1][:n]) & set(range(nb)))


@pytest.mark.parametrize("bpc", [2, 3, 8])
def test_project_band_loop_of_a_cta(sho, bpc):
    """A CTA of sho_project may project several consecutive bands with the tables it sampled once (the launch picks
    that for many bands of a small grid: the paper's workload).  Forced here on small inputs through the plan's
    test knob (sho_plan_set_option): band counts that are and are not multiples of the group, real and complex data, remainder rows."""
    for w in (workloads.make_paper(5, "r64", size="small"), workloads.make(5, size="small"), workloads.make(2, size="small")):
        for nb in (w.nbands, 5):
            w.nbands = nb
            run_case(sho, w, stored=False, options={"project_bands_per_cta": bpc})
    # the grouping changes which CTA computes a band, not how: bit-identical coefficients
    import torch
    w = workloads.make(5, size="small")
    plan = sho.plan_for(w)
    try:
        psi = _dev(w.psi())
        c_grouped = plan.set_option("project_bands_per_cta", bpc).project(psi).clone()
        c_single = plan.set_option("project_bands_per_cta", 1).project(psi)
        torch.cuda.synchronize()
        assert torch.equal(torch.view_as_real(c_grouped), torch.view_as_real(c_single))
    finally:
        plan.close()


@pytest.mark.parametrize("k,dtype", [(3, None), (4, None), (4, "r32"), (5, None), ("paper", "r64"), ("paper", "r32")])
def test_full_size_config_sampled(sho, k, dtype):
    """BASELINE.json config k at its full size, in the launch configuration bench.py times (all bands, device
    inputs from a seeded torch generator), sampled as SURVEY 8(d) asks:
      project: >= 64 (atom, band) pairs -- atoms whose box wraps on every axis, on none, the smallest and the
               largest sigma -- over 8 bands including interior ones, each computed by the oracle's direct sum;
      stored-projector project (cfg 3, the config it is timed on): the same pairs;
      add:     into a NON-ZERO psi: four full z-planes (0, Nz-1, the first plane of the second tile layer, a
               middle plane) for 8 bands, plus 4096 random points for ALL bands, every value computed
               point-wise by the oracle.  Norms of reading A13 over the samples."""
    import torch
    w = workloads.make_paper(5, dtype) if k == "paper" else workloads.make(k, dtype=dtype)   # paper: 8 bands per CTA
    if dtype in ("r32", "r64"):
        w.kfrac = None
    tol = TOL[w.dtype]
    wide = np.complex128 if w.is_complex else np.float64
    tdt = {"r64": torch.float64, "c128": torch.complex128, "r32": torch.float32, "c64": torch.complex64}[w.dtype]
    plan = sho.plan_for(w)
    try:
        boxes = _oracle_boxes(w)
        assert np.array_equal(plan.boxes(), boxes), "integer box ranges differ from the oracle"
        gen = torch.Generator(device="cuda")
        gen.manual_seed(w.seed)
        shape = (w.nbands, w.ng[2], w.ng[1], w.ng[0])
        psi = torch.randn(shape, dtype=tdt, device="cuda", generator=gen)
        c_gpu = plan.project(psi)
        torch.cuda.synchronize()
        # ---- project: sampled pairs ----
        atoms = _sample_atoms(w, boxes)
        bsel = _sample_bands(w.nbands)
        pairs = [(a, b) for a in atoms for b in bsel]
        assert len(pairs) >= 64 and len(bsel) >= 8
        bands = {b: psi[b].cpu().numpy().astype(wide) for b in bsel}
        pa, pb = np.array([q[0] for q in pairs]), np.array([q[1] for q in pairs])
        ref = oracle.project_pairs(w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax, bands, pa, pb, w.nbands,
                                   w.is_complex, w.rcut_sigma)
        norm = np.array([np.sqrt(w.h ** 3 * np.sum(np.abs(bands[int(b)]) ** 2)) for b in pb])
        ia, ib = torch.as_tensor(pa, device="cuda"), torch.as_tensor(pb, device="cuda")
        got = c_gpu[ia, ib].cpu().numpy().astype(wide)
        err = (np.abs(got - ref) / norm[:, None]).max()
        assert err <= tol, "project parity at full size: %.3e > %.1e" % (err, tol)
        # ---- stored-projector baseline at the size it is timed on (cfg 3: 53 GB of tables) ----
        if k == 3:
            tb = plan.tables()
            c_sto = plan.project_stored(tb, psi)
            torch.cuda.synchronize()
            got = c_sto[ia, ib].cpu().numpy().astype(wide)
            tb.close()
            err = (np.abs(got - ref) / norm[:, None]).max()
            assert err <= tol, "stored-projector parity at full size: %.3e > %.1e" % (err, tol)
            del c_sto
        # ---- add into the non-zero psi: full planes of 8 bands + random points of all bands ----
        coeff = torch.randn((w.natoms, w.nbands, plan.nsho), dtype=tdt, device="cuda", generator=gen)
        psi0 = psi.clone()
        plan.add(coeff, psi)
        torch.cuda.synchronize()
        coeff_h = coeff.cpu().numpy().astype(wide)
        Nx, Ny, Nz = w.ng
        worst = 0.0
        for jz in (0, Nz - 1, 8, Nz // 2 + 3):
            yy, xx = np.meshgrid(np.arange(Ny), np.arange(Nx), indexing="ij")
            pts = np.stack([xx.ravel(), yy.ravel(), np.full(xx.size, jz)], axis=1)
            inc = oracle.add_points_bands(w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax, coeff_h, pts, bsel,
                                          w.rcut_sigma)                                   # [Ny*Nx][8]
            tb_ = torch.as_tensor(bsel, device="cuda")
            refp = psi0[tb_, jz].cpu().numpy().astype(wide).reshape(len(bsel), -1).T + inc
            gotp = psi[tb_, jz].cpu().numpy().astype(wide).reshape(len(bsel), -1).T
            e = (np.abs(gotp - refp).max(axis=0) / np.abs(refp).max(axis=0)).max()
            worst = max(worst, float(e))
            assert e <= tol, "add parity at full size, plane z = %d: %.3e > %.1e" % (jz, e, tol)
        rng = np.random.default_rng(w.seed)
        pts = np.stack([rng.integers(0, w.ng[d], 4096) for d in range(3)], axis=1)
        allb = np.arange(w.nbands)
        inc = oracle.add_points_bands(w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax, coeff_h, pts, allb, w.rcut_sigma)
        iz, iy, ix = (torch.as_tensor(pts[:, d], device="cuda") for d in (2, 1, 0))
        refp = psi0[:, iz, iy, ix].cpu().numpy().astype(wide).T + inc
        gotp = psi[:, iz, iy, ix].cpu().numpy().astype(wide).T
        e = (np.abs(gotp - refp).max(axis=0) / np.abs(refp).max(axis=0)).max()
        assert e <= tol, "add parity at full size, random points of all bands: %.3e > %.1e" % (e, tol)
    finally:
        plan.close()


def test_cfg2_at_its_stated_size_in_full(sho):
    """"Parity: full at cfg 1-3".  Config 2 as BASELINE.json states it (96^3 periodic, 32 atoms, numax 5,
    16 bands): project, stored project, add, stored-1D and stored add compared with the oracle on EVERY element."""
    w = workloads.make(2)
    assert w.ng == (96, 96, 96) and w.natoms == 32 and w.nbands == 16 and w.numax == 5
    run_case(sho, w)


def test_cfg3_projection_at_its_stated_size_in_full(sho):
    """Config 3 as stated (128^3 periodic, 256 atoms, numax 7, 32 bands): all 8192 x 120 coefficients against the
    oracle's direct sum (2e11 multiply-adds on the host cores, about a minute).  The add-back of this config is
    covered by the sampled full-size test above (planes and points computed point-wise by the oracle)."""
    import torch
    w = workloads.make(3)
    assert w.ng == (128, 128, 128) and w.natoms == 256 and w.nbands == 32 and w.numax == 7
    plan = sho.plan_for(w)
    try:
        assert np.array_equal(plan.boxes(), _oracle_boxes(w)), "integer box ranges differ from the oracle"
        psi = w.psi()
        c_gpu = plan.project(_dev(psi))
        torch.cuda.synchronize()
        check_project(sho, w, psi, c_gpu.cpu().numpy(), TOL[w.dtype])
    finally:
        plan.close()


def _atoms_touching(w, boxes, pts):
    """Atoms whose box (any periodic image) contains at least one of the grid points pts[n][3] = (jx, jy, jz)."""
    hit = np.ones((w.natoms, len(pts)), bool)
    for d in range(3):
        N = w.ng[d]
        on_axis = np.zeros((w.natoms, len(pts)), bool)
        for m in (-2, -1, 0, 1, 2) if w.periodic[d] else (0,):
            i = pts[:, d][None, :] + m * N
            on_axis |= (i >= boxes[:, d, 0][:, None]) & (i <= boxes[:, d, 1][:, None])
        hit &= on_axis
    return np.nonzero(hit.any(axis=1))[0]


def test_apply_host_at_cfg5_full_size_with_the_natural_chunk_rule(sho):
    """sho_apply_host -- the call bench.py's end-to-end number is measured through -- at config 5's full size with the
    library's own chunk rule (no "host_chunk_bands" option: one 113 MB band per chunk, 64 chunks through the three-slot
    ring).  The three steps of PAPER.md:187-190 are recomputed by the oracle for two bands at the points of one
    8 x 64 x 8 block of the grid and of a 4 x 4 x 4 block around the cell corner (every image wraps there, Bloch
    phases on all axes): project_pairs for every atom whose box touches those points, dmul, add_points_bands."""
    import torch
    w = workloads.make(5)
    assert w.ng == (192, 192, 192) and w.natoms == 1024 and w.nbands == 64 and w.dtype == "c128"
    plan = sho.plan_for(w)
    try:
        boxes = _oracle_boxes(w)
        assert np.array_equal(plan.boxes(), boxes)
        Nx, Ny, Nz = w.ng
        bsel = [17, 63]
        gen = torch.Generator(device="cuda")
        gen.manual_seed(w.seed + 5)
        host = torch.empty((w.nbands, Nz, Ny, Nx), dtype=torch.complex128, pin_memory=True)
        bands = {}
        for b in range(w.nbands):
            band = torch.randn((Nz, Ny, Nx), dtype=torch.complex128, device="cuda", generator=gen)
            host[b].copy_(band)
            if b in bsel:
                bands[b] = band.cpu().numpy()
        del band
        torch.cuda.synchronize()
        Dm = w.dmatrix(plan.nsho)
        plan.apply_host(Dm, host)
        # ---- the oracle on the sampled points ----
        blk = np.stack(np.meshgrid(np.arange(40, 48), np.arange(64, 128), np.arange(16, 24), indexing="ij"), -1).reshape(-1, 3)
        edge = np.array([Nx - 2, Nx - 1, 0, 1])
        cor = np.stack(np.meshgrid(edge, edge, edge, indexing="ij"), -1).reshape(-1, 3)
        pts = np.concatenate([blk, cor]).astype(np.int32)
        atoms = _atoms_touching(w, boxes, pts)
        assert 20 <= len(atoms) <= 400
        pa = np.repeat(atoms, len(bsel))
        pb = np.tile(np.array(bsel), len(atoms))
        geo = (w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax)
        c = oracle.project_pairs(*geo, bands, pa, pb, w.nbands, True, w.rcut_sigma)             # [pairs][N_SHO]
        c = c.reshape(len(atoms), len(bsel), plan.nsho)
        d = oracle.dmul(np.ascontiguousarray(Dm[atoms]), c)
        coeff = np.zeros((w.natoms, w.nbands, plan.nsho), np.complex128)                       # atoms that do not touch
        coeff[np.ix_(atoms, bsel)] = d                                                         # the points add nothing there
        inc = oracle.add_points_bands(*geo, coeff, pts, bsel, w.rcut_sigma)                      # [npts][2]
        for i, b in enumerate(bsel):
            ref = bands[b][pts[:, 2], pts[:, 1], pts[:, 0]] + inc[:, i]
            got = host[b].numpy()[pts[:, 2], pts[:, 1], pts[:, 0]]
            assert np.abs(inc[:, i]).max() > 1e-3 * np.abs(ref).max()                           # the action did something
            err = np.abs(got - ref).max() / np.abs(ref).max()
            assert err <= 1e-12, "sho_apply_host at cfg 5, band %d: %.3e > 1e-12" % (b, err)
    finally:
        plan.close()


def test_dmul_and_transform_at_cfg5_full_size_in_full(sho):
    """Step (2) d = D c and the spherical transform (eq. (10)-(11)) on all of config
    5's 1024 x 64 x 220 complex coefficients against oracle.dmul, every element."""
    import torch
    w = workloads.make(5)
    plan = sho.plan_for(w)
    try:
        rng = np.random.default_rng(55)
        D = rng.standard_normal((w.natoms, plan.nsho, plan.nsho)) / np.sqrt(plan.nsho)           # not symmetric
        c = w.coeff(plan.nsho)
        ref = oracle.dmul(D, c)
        d_c = _dev(c)
        out = plan.dmul(_dev(D), d_c)
        torch.cuda.synchronize()
        assert np.abs(out.cpu().numpy() - ref).max() <= 1e-12 * np.abs(ref).max()
        del out, D
        Uo = oracle.umatrix(w.numax)
        ref = oracle.dmul(np.ascontiguousarray(np.broadcast_to(Uo, (w.natoms,) + Uo.shape)), c)
        out = plan.transform(_dev(sho.umatrix(w.numax)), d_c)
        torch.cuda.synchronize()
        assert np.abs(out.cpu().numpy() - ref).max() <= 1e-12 * np.abs(ref).max()
    finally:
        plan.close()


def test_band_fastest_layout_at_the_papers_full_size(sho):
    """sho_project_bf / sho_add_bf on the paper's own workload at full size (64^3, 665 atoms, 1024 bands, psi_bf of
    2.1 GB, chunks of 64 bands): sampled (atom, band) pairs against the oracle's direct sum, and the add-back at 2048
    random points of ALL bands computed point-wise by the oracle."""
    import torch
    w = workloads.make_paper(5, "r64")
    plan = sho.plan_for(w)
    try:
        boxes = _oracle_boxes(w)
        gen = torch.Generator(device="cuda")
        gen.manual_seed(w.seed + 1)
        psi = torch.randn((w.nbands, w.ng[2], w.ng[1], w.ng[0]), dtype=torch.float64, device="cuda", generator=gen)
        psi_bf = psi.permute(1, 2, 3, 0).contiguous()
        c_bf = plan.project_bf(psi_bf)
        torch.cuda.synchronize()
        atoms = _sample_atoms(w, boxes)
        bsel = _sample_bands(w.nbands)
        pa = np.repeat(np.array(atoms), len(bsel))
        pb = np.tile(np.array(bsel), len(atoms))
        bands = {b: psi[b].cpu().numpy() for b in bsel}
        ref = oracle.project_pairs(w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax, bands, pa, pb, w.nbands,
                                   False, w.rcut_sigma)
        norm = np.array([np.sqrt(w.h ** 3 * np.sum(bands[int(b)] ** 2)) for b in pb])
        got = c_bf[torch.as_tensor(pa, device="cuda"), torch.as_tensor(pb, device="cuda")].cpu().numpy()
        err = (np.abs(got - ref) / norm[:, None]).max()
        assert err <= 1e-12, "sho_project_bf at the paper's full size: %.3e" % err
        coeff = torch.randn((w.natoms, w.nbands, plan.nsho), dtype=torch.float64, device="cuda", generator=gen)
        del psi
        before = psi_bf.clone()
        plan.add_bf(coeff, psi_bf)
        torch.cuda.synchronize()
        rng = np.random.default_rng(w.seed)
        pts = np.stack([rng.integers(0, w.ng[d], 2048) for d in range(3)], axis=1)
        inc = oracle.add_points_bands(w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax, coeff.cpu().numpy(), pts,
                                      np.arange(w.nbands), w.rcut_sigma)                          # [npts][nbands]
        iz, iy, ix = (torch.as_tensor(pts[:, d], device="cuda") for d in (2, 1, 0))
        refp = before[iz, iy, ix].cpu().numpy() + inc
        gotp = psi_bf[iz, iy, ix].cpu().numpy()
        e = (np.abs(gotp - refp).max(axis=0) / np.abs(refp).max(axis=0)).max()
        assert e <= 1e-12, "sho_add_bf at the paper's full size: %.3e" % e
    finally:
        plan.close()


@pytest.mark.parametrize("case", range(24))
def test_seeded_random_geometries(sho, case):
    """Seeded random small problems, every one compared with the oracle in full (project, add, stored variants): odd
    grid dims, any mix of periodic and isolated axes, atoms inside, on the faces and well outside the cell, sigma such
    that a box is at most as wide as the cell, numax 0 .. 11 (every K-step count, the remainder rows of numax 8, 9 and
    their shared K step in the add), 1 .. 5 bands, all four element types, random Bloch phases for complex data."""
    rng = np.random.default_rng(20260000 + case)
    ng = tuple(int(v) for v in rng.integers(9, 41, 3))
    periodic = tuple(int(v) for v in rng.integers(0, 2, 3))
    h = float(rng.choice([0.2, 0.25, 0.3]))
    numax = int(rng.integers(0, 12)) if case % 3 else int(rng.choice([8, 9]))
    dtype = ["r64", "c128", "r32", "c64"][case % 4]
    natoms = int(rng.integers(1, 6))
    L = np.array(ng) * h
    pos = (rng.random((natoms, 3)) * 2.0 - 0.5) * L                    # from half a cell before to half a cell behind
    smax = 0.999 * (min(ng) - 1) * h / 12.0                            # 6 sigma on both sides fit the narrowest axis
    sigma = rng.uniform(0.45 * smax, smax, natoms)
    kfrac = None
    if dtype in ("c128", "c64"):
        kfrac = tuple(float(k) if per else 0.0 for k, per in zip(rng.uniform(-0.5, 0.5, 3), periodic))
    w = _custom(ng, periodic, pos, sigma, numax, int(rng.integers(1, 6)), dtype=dtype, h=h, kfrac=kfrac, seed=500 + case)
    run_case(sho, w, stored=(case % 2 == 0))


def test_box_exactly_as_wide_as_the_cell(sho):
    # periodic box of exactly N points on x (every grid point once, one wrap)
    ng = (24, 40, 40)
    w = _custom(ng, (1, 1, 1), [[1.13, 5.0, 5.0]], [0.4834], 3, 2, h=0.25)
    lo, hi, _ = oracle.box(w.ng, w.h, w.periodic, w.pos[0], w.sigma[0], 6.0)
    assert hi[0] - lo[0] + 1 == 24
    run_case(sho, w)


def test_box_wider_than_cell_is_reported_unsupported(sho):
    w = _custom((16, 16, 16), (1, 1, 1), [[1.0, 1.0, 1.0]], [1.0], 2, 1)
    with pytest.raises(sho.ShoError) as ei:
        sho.plan_for(w)
    assert ei.value.status == 2


def test_unaligned_psi_pointer(sho):
    # psi starting 8 bytes into an allocation: the 16-byte vector path must not be taken
    import torch
    w = workloads.make(2, size="small")
    plan = sho.plan_for(w)
    psi = w.psi()
    buf = torch.zeros(psi.size + 1, dtype=torch.float64, device="cuda")
    view = buf[1:].view(psi.shape)
    view.copy_(torch.from_numpy(psi))
    c = plan.project(view)
    torch.cuda.synchronize()
    check_project(sho, w, psi, c.cpu().numpy(), 1e-12)
    coeff = w.coeff(plan.nsho)
    plan.add(_dev(coeff), view)
    torch.cuda.synchronize()
    ref = oracle.add(w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax, coeff, psi)
    assert np.abs(view.cpu().numpy() - ref).max() <= 1e-12 * np.abs(ref).max()
    plan.close()


def test_add_is_bit_reproducible(sho):
    import torch
    w = workloads.make(4, size="small")
    plan = sho.plan_for(w)
    c = _dev(w.coeff(plan.nsho))
    outs = []
    for _ in range(3):
        psi = torch.zeros((w.nbands, w.ng[2], w.ng[1], w.ng[0]), dtype=torch.float64, device="cuda")
        plan.add(c, psi)
        torch.cuda.synchronize()
        outs.append(psi)
    assert torch.equal(outs[0], outs[1]) and torch.equal(outs[0], outs[2])
    plan.close()


@pytest.mark.parametrize("name", ["cfg2-small", "cfg5-small", "ragged"])
def test_no_write_outside_the_callers_buffers(sho, name):
    """compute-sanitizer is closed on this pool (it cannot attach to a process there), so out-of-bounds WRITES are caught here:
    psi and coeff live inside larger allocations whose guard zones (64 KB on each side, a NaN bit pattern) must come
    back untouched from project, add, the stored-projector project and the fused action; reads outside the buffers
    would hit NaNs and fail the finiteness / parity checks of the other tests."""
    import torch
    if name == "ragged":
        rng = np.random.default_rng(3)
        ng = (33, 37, 29)
        w = _custom(ng, (1, 0, 1), rng.uniform(0, 1, (5, 3)) * np.array(ng) * 0.25, rng.uniform(0.35, 0.6, 5), 9, 3,
                    dtype="c128", kfrac=(0.1, 0.0, 0.3))
    else:
        w = workloads.make(int(name[3]), size="small")
    plan = sho.plan_for(w)
    G = 8192                                     # guard elements (64 KB of fp64)
    tdt = torch.complex128 if w.is_complex else torch.float64

    def guarded(shape):
        n = int(np.prod(shape))
        buf = torch.full((n + 2 * G,), complex("nan+nanj") if w.is_complex else float("nan"), dtype=tdt, device="cuda")
        return buf, buf[G:G + n].view(shape)

    def intact(buf, n):
        g = torch.view_as_real(buf).reshape(-1) if w.is_complex else buf
        k = 2 if w.is_complex else 1
        return bool(torch.isnan(g[:G * k]).all()) and bool(torch.isnan(g[(G + n) * k:]).all())

    try:
        psi_h = w.psi()
        if w.psi_dist == "zero":
            psi_h = workloads.Workload(**{**w.__dict__, "psi_dist": "normal"}).psi()
        pbuf, psi = guarded(psi_h.shape)
        psi.copy_(torch.from_numpy(psi_h))
        cbuf, c = guarded((w.natoms, w.nbands, plan.nsho))
        c.zero_()
        plan.project(psi, c)
        plan.add(c, psi)
        tb = plan.tables()
        plan.project_stored(tb, psi, c)
        if hasattr(plan, "apply"):
            D = torch.from_numpy(np.tile(np.eye(plan.nsho), (w.natoms, 1, 1))).cuda()
            plan.apply(D, psi, c)
        torch.cuda.synchronize()
        tb.close()
        assert intact(pbuf, psi.numel()), "a kernel wrote outside psi"
        assert intact(cbuf, c.numel()), "a kernel wrote outside coeff"
        assert bool(torch.isfinite(torch.view_as_real(psi) if w.is_complex else psi).all())
        assert bool(torch.isfinite(torch.view_as_real(c) if w.is_complex else c).all())
    finally:
        plan.close()


@pytest.mark.parametrize("k", [4, 5])
def test_project_and_add_are_bit_reproducible_under_load(sho, k):
    """Stand-in for racecheck (closed on this pool): both kernels are deterministic by construction (fixed
    summation order, no atomics), so ANY shared-memory race shows up as a run-to-run difference.  Five runs,
    half of them with a second stream hammering the GPU to perturb the warp schedule."""
    import torch
    w = workloads.make(k, size="small")
    plan = sho.plan_for(w)
    psi_h = workloads.Workload(**{**w.__dict__, "psi_dist": "normal"}).psi()
    c_h = w.coeff(plan.nsho)
    side = torch.cuda.Stream()
    junk = torch.randn(2048, 2048, device="cuda")
    ref = None
    for it in range(5):
        if it % 2:
            with torch.cuda.stream(side):
                for _ in range(20):
                    junk = junk @ junk * 1e-3
        psi = _dev(psi_h)
        cc = plan.project(psi)
        out = _dev(psi_h)
        plan.add(_dev(c_h), out)
        torch.cuda.synchronize()
        cur = (cc.clone(), out.clone())
        if ref is None:
            ref = cur
        assert torch.equal(ref[0], cur[0]) and torch.equal(ref[1], cur[1]), "run %d differs bit-wise from run 0" % it
    plan.close()


def test_stored_projection_is_bit_reproducible(sho):
    # its K segments are added in a fixed order through a turnstile, not by atomicAdd
    import torch
    w = workloads.make(3, size="small")
    plan = sho.plan_for(w)
    psi = _dev(w.psi())
    tb = plan.tables()
    outs = [plan.project_stored(tb, psi).clone() for _ in range(4)]
    torch.cuda.synchronize()
    tb.close()
    plan.close()
    assert all(torch.equal(outs[0], o) for o in outs[1:])


def test_stored_projections_sharing_one_tables_object_on_two_streams(sho):
    """The hand-over counters of sho_project_stored live in the tables object: launches that share it are chained on
    the device by the library, so issuing them on two streams at once must give what one stream gives (bit for bit),
    not a race on the counters (wrong sums or a hang)."""
    import torch
    w = workloads.make(2)                                  # full size: 3.3 GB of tables, kernels of about a millisecond
    plan = sho.plan_for(w)
    psi_a = _dev(w.psi())
    psi_b = psi_a.flip(0).contiguous()                     # the same bands in another order: other data per launch
    tb = plan.tables()
    try:
        ref_a = plan.project_stored(tb, psi_a).clone()
        ref_b = plan.project_stored(tb, psi_b).clone()
        torch.cuda.synchronize()
        assert torch.equal(ref_a, ref_b.flip(1))
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        outs_a = [plan.new_coeff(w.nbands, psi_a.device) for _ in range(6)]
        outs_b = [plan.new_coeff(w.nbands, psi_a.device) for _ in range(6)]
        for oa, ob in zip(outs_a, outs_b):
            plan.project_stored(tb, psi_a, oa, stream=s1)
            plan.project_stored(tb, psi_b, ob, stream=s2)
        torch.cuda.synchronize()
        assert all(torch.equal(ref_a, o) for o in outs_a)
        assert all(torch.equal(ref_b, o) for o in outs_b)
    finally:
        tb.close()
        plan.close()


def test_host_buffer_entry_points(sho):
    w = workloads.make(3, size="small")
    plan = sho.plan_for(w)
    psi = w.psi()
    c = np.zeros((w.natoms, w.nbands, plan.nsho))
    plan.project_host(psi, c)
    check_project(sho, w, psi, c, 1e-12)
    coeff = w.coeff(plan.nsho)
    out = psi.copy()
    plan.add_host(coeff, out)
    ref = oracle.add(w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax, coeff, psi)
    assert np.abs(out - ref).max() <= 1e-12 * np.abs(ref).max()
    plan.close()


@pytest.mark.parametrize("k,chunk", [(3, "2"), (3, "3"), (5, "1"), (5, "2")])
def test_host_buffer_calls_pipeline_band_chunks(sho, k, chunk):
    # the *_host calls copy and compute band chunks on three streams; force several (ragged) chunks
    w = workloads.make(k, size="small")
    wide = np.complex128 if w.is_complex else np.float64
    plan = sho.plan_for(w)
    try:
        plan.set_option("host_chunk_bands", int(chunk))
        psi = w.psi()
        c = np.zeros((w.natoms, w.nbands, plan.nsho), dtype=psi.dtype)
        plan.project_host(psi, c)
        check_project(sho, w, psi, c, TOL[w.dtype])
        coeff = w.coeff(plan.nsho)
        out = psi.copy()
        plan.add_host(coeff, out)
        ref = oracle.add(w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax, coeff.astype(wide), psi.astype(wide))
        assert np.abs(out - ref).max() <= TOL[w.dtype] * np.abs(ref).max()
    finally:
        plan.close()


# ------------------------------------------------------------------------------------------------
# step (2) d = D c and the three-step non-local action


@pytest.mark.parametrize("k,dtype", [(1, None), (2, None), (3, "r32"), (4, None), (5, None), (5, "c64")])
def test_dmul_and_apply_match_the_oracle(sho, k, dtype):
    """sho_dmul against oracle.dmul (not symmetric D: a transposed product fails), in place and out of place;
    sho_apply against add(dmul(project(psi))) of the oracle; sho_apply_host (one upload of psi) against the same."""
    import torch
    w = workloads.make(k, size="small", dtype=dtype)
    if dtype in ("r32", "r64"):
        w.kfrac = None
    tol = TOL[w.dtype]
    wide = np.complex128 if w.is_complex else np.float64
    plan = sho.plan_for(w)
    try:
        rng = np.random.default_rng(k)
        D = rng.standard_normal((w.natoms, plan.nsho, plan.nsho)) / np.sqrt(plan.nsho)
        c = w.coeff(plan.nsho)
        ref = oracle.dmul(D, c.astype(wide))
        d_D = _dev(D)
        out = plan.dmul(d_D, _dev(c))
        torch.cuda.synchronize()
        scale = np.abs(ref).max()
        assert np.abs(out.cpu().numpy().astype(wide) - ref).max() <= tol * scale
        inpl = _dev(c)
        plan.dmul(d_D, inpl, inpl)
        torch.cuda.synchronize()
        assert torch.equal(inpl, out), "in-place sho_dmul differs from out-of-place"
        # the whole action with the workload's symmetric D
        Dm = w.dmatrix(plan.nsho)
        psi = w.psi()
        if w.psi_dist == "zero":
            psi = workloads.Workload(**{**w.__dict__, "psi_dist": "normal"}).psi()
        geo = (w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax)
        c_ref = oracle.project(*geo, psi.astype(wide), w.rcut_sigma)
        psi_ref = oracle.add(*geo, oracle.dmul(Dm, c_ref), psi.astype(wide), w.rcut_sigma)
        scale = np.maximum(np.abs(psi_ref).max(axis=(1, 2, 3)), 1e-300)
        d_psi = _dev(psi)
        work = plan.new_coeff(w.nbands)
        plan.apply(_dev(Dm), d_psi, work)
        torch.cuda.synchronize()
        err = (np.abs(d_psi.cpu().numpy().astype(wide) - psi_ref).max(axis=(1, 2, 3)) / scale).max()
        assert err <= tol, "sho_apply parity: %.3e > %.1e" % (err, tol)
        d_ref = oracle.dmul(Dm, c_ref)
        norm = _psi_norm(psi, w.h)
        errd = (np.abs(work.cpu().numpy().astype(wide) - d_ref) / norm[None, :, None]).max()
        assert errd <= tol * max(1.0, np.abs(Dm).sum(axis=2).max()), "coeff_work must hold d = D c on return"
        host = psi.copy()
        plan.apply_host(Dm, host)
        err = (np.abs(host.astype(wide) - psi_ref).max(axis=(1, 2, 3)) / scale).max()
        assert err <= tol, "sho_apply_host parity: %.3e > %.1e" % (err, tol)
    finally:
        plan.close()


@pytest.mark.parametrize("chunk", ["1", "2"])
def test_apply_host_pipelines_band_chunks_through_a_bounded_ring(sho, chunk):
    # 5 bands in chunks of 1 or 2: more chunks than the three ring slots, so slots are reused
    rng = np.random.default_rng(9)
    ng = (24, 40, 16)
    w = _custom(ng, (1, 1, 1), rng.uniform(0, 1, (6, 3)) * np.array(ng) * 0.25, rng.uniform(0.3, 0.36, 6), 5, 5, rc=4.0)
    plan = sho.plan_for(w)
    try:
        plan.set_option("host_chunk_bands", int(chunk))
        Dm = w.dmatrix(plan.nsho)
        psi = w.psi()
        geo = (w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax)
        c_ref = oracle.project(*geo, psi, w.rcut_sigma)
        psi_ref = oracle.add(*geo, oracle.dmul(Dm, c_ref), psi, w.rcut_sigma)
        host = psi.copy()
        plan.apply_host(Dm, host)
        assert np.abs(host - psi_ref).max() <= 1e-12 * np.abs(psi_ref).max()
        c = np.zeros((w.natoms, w.nbands, plan.nsho))
        plan.project_host(psi, c)
        check_project(sho, w, psi, c, 1e-12)
        out = psi.copy()
        plan.add_host(c_ref, out)
        ref = oracle.add(*geo, c_ref, psi, w.rcut_sigma)
        assert np.abs(out - ref).max() <= 1e-12 * np.abs(ref).max()
    finally:
        plan.close()


# ------------------------------------------------------------------------------------------------
# the paper's own workload (sec. 6) and its band-fastest psi layout


@pytest.mark.parametrize("numax,dtype", [(0, "r64"), (2, "r64"), (5, "r64"), (4, "r32")])
def test_paper_workload_small(sho, numax, dtype):
    """PAPER.md:369-377 at 24^3 points / 16 bands: isolated domain, fcc atoms of which most sit outside the grid
    with a clipped region; full comparison with the oracle."""
    run_case(sho, workloads.make_paper(numax, dtype, size="small"))


@pytest.mark.parametrize("dtype,nb,wb", [("r64", 16, 16), ("r64", 7, 2), ("r32", 5, 1), ("c128", 3, 2)])
def test_band_fastest_layout_entry_points(sho, dtype, nb, wb):
    """sho_project_bf / sho_add_bf on psi_bf[Nz][Ny][Nx][nbands] against the oracle on the transposed
    data, with workspaces of wb bands (several chunks, ragged last chunk, odd band counts)."""
    import torch
    w = workloads.make_paper(3, dtype, size="small") if dtype != "c128" else workloads.make(5, size="small")
    w.nbands = nb
    tol = TOL[w.dtype]
    wide = np.complex128 if w.is_complex else np.float64
    plan = sho.plan_for(w)
    try:
        psi = w.psi()                                              # [nb][Nz][Ny][Nx]
        psi_bf = _dev(np.ascontiguousarray(np.moveaxis(psi, 0, 3)))
        work = torch.empty((wb, w.ng[2], w.ng[1], w.ng[0]), dtype=psi_bf.dtype, device="cuda")
        c = plan.project_bf(psi_bf, work=work)
        torch.cuda.synchronize()
        check_project(sho, w, psi, c.cpu().numpy(), tol)
        coeff = w.coeff(plan.nsho)
        plan.add_bf(_dev(coeff), psi_bf, work=work)
        torch.cuda.synchronize()
        ref = oracle.add(w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax, coeff.astype(wide), psi.astype(wide), w.rcut_sigma)
        got = np.moveaxis(psi_bf.cpu().numpy(), 3, 0).astype(wide)
        scale = np.abs(ref).max(axis=(1, 2, 3))
        assert (np.abs(got - ref).max(axis=(1, 2, 3)) / scale).max() <= tol
        with pytest.raises(sho.ShoError):
            plan.project_bf(psi_bf, work=torch.empty(8, dtype=psi_bf.dtype, device="cuda"))
    finally:
        plan.close()


@pytest.mark.parametrize("k,dtype", [(2, None), (5, None), (4, "r32")])
def test_transform_to_the_spherical_representation(sho, k, dtype):
    """sho_transform with the library's U against the oracle's U applied by the oracle's dmul (f4),
    and back with the transpose."""
    import torch
    w = workloads.make(k, size="small", dtype=dtype)
    if dtype in ("r32", "r64"):
        w.kfrac = None
    wide = np.complex128 if w.is_complex else np.float64
    plan = sho.plan_for(w)
    try:
        c = w.coeff(plan.nsho)
        Uo = oracle.umatrix(w.numax)
        ref = oracle.dmul(np.tile(Uo, (w.natoms, 1, 1)), c.astype(wide))
        U = sho.umatrix(w.numax)
        d_c = _dev(c)
        out = plan.transform(_dev(U), d_c)
        back = plan.transform(_dev(np.ascontiguousarray(U.T)), out)
        torch.cuda.synchronize()
        tol = TOL[w.dtype]
        assert np.abs(out.cpu().numpy().astype(wide) - ref).max() <= tol * np.abs(ref).max()
        assert np.abs(back.cpu().numpy().astype(wide) - c.astype(wide)).max() <= (1e-12 if tol < 1e-6 else 1e-5) * np.abs(c).max()
    finally:
        plan.close()


def test_wrong_arguments_raise(sho):
    import torch
    w = workloads.make(1)
    plan = sho.plan_for(w)
    with pytest.raises(ValueError):
        plan.project(torch.zeros((1, 32, 32, 32), dtype=torch.float32, device="cuda"))
    with pytest.raises(ValueError):
        plan.project(torch.zeros((1, 32, 32, 31), dtype=torch.float64, device="cuda"))
    with pytest.raises(sho.ShoError):
        sho.Plan((32, 32, 32), -1.0, (0, 0, 0), w.pos, w.sigma, 3)
    with pytest.raises(sho.ShoError):
        sho.Plan((32, 32, 32), 0.25, (0, 0, 0), w.pos, w.sigma, 16)
    with pytest.raises(sho.ShoError):
        sho.Plan((32, 32, 32), 0.25, (1, 1, 1), w.pos, w.sigma, 3, "r64", kfrac=(0.1, 0, 0))
    for key, value in (("no_such_option", 1), ("project_bands_per_cta", 9), ("project_bands_per_cta", -1), ("host_chunk_bands", -2)):
        with pytest.raises(sho.ShoError):
            plan.set_option(key, value)
    plan.set_option("project_bands_per_cta", 0).set_option("host_chunk_bands", 0)
    plan.close()
