"""Pins for the CPU oracle (oracle/sho_oracle.c) against things OTHER than itself.

Each test is chosen so that a plausible mistake in the oracle (dropped h^3, wrong Hermite sign or
normalisation, transposed axes, wrong wrap / Bloch-phase sign, off-by-one box edge, wrong coefficient
order) fails at least one of them.  References used here: values printed in the paper
(tests/golden/*.txt), scipy's Hermite polynomials and quadrature (library routines), closed forms,
and invariants.  SURVEY.md 8(c) pins P1-P8.  CPU only.
"""
import math
import warnings

import numpy as np
import pytest
from scipy import integrate, special

import oracle

# ----------------------------------------------------------------------------------------------
# independent helpers (scipy Hermite; no oracle arithmetic)


def lib_phi(n, u, sigma):
    """Normalised Hermite-Gauss function from scipy's H_n (library routine)."""
    xi = np.asarray(u, dtype=np.float64) / sigma
    norm = 1.0 / math.sqrt(2.0 ** n * math.factorial(n) * math.sqrt(math.pi) * sigma)
    return norm * special.eval_hermite(n, xi) * np.exp(-0.5 * xi * xi)


def lib_ranges(ng, h, periodic, pos, sigma, rc):
    lo = np.ceil((np.asarray(pos) - rc * sigma) / h).astype(int)
    hi = np.floor((np.asarray(pos) + rc * sigma) / h).astype(int)
    for d in range(3):
        if not periodic[d]:
            lo[d] = max(lo[d], 0)
            hi[d] = min(hi[d], ng[d] - 1)
    return lo, hi


def separable_project(ng, h, periodic, kfrac, pos, sigma, numax, psi, rc):
    """Separable x->y->z contraction with numpy einsum and scipy 1D tables (pin P2's other side)."""
    na, nb = len(sigma), psi.shape[0]
    out = np.zeros((na, nb, oracle.nsho(numax)), dtype=psi.dtype)
    for a in range(na):
        lo, hi = lib_ranges(ng, h, periodic, pos[a], sigma[a], rc)
        if np.any(hi < lo):
            continue
        idx = [np.arange(lo[d], hi[d] + 1) for d in range(3)]
        tab = [np.stack([lib_phi(n, idx[d] * h - pos[a][d], sigma[a]) for n in range(numax + 1)]) for d in range(3)]
        sub = psi[:, np.mod(idx[2], ng[2])[:, None, None], np.mod(idx[1], ng[1])[None, :, None],
                  np.mod(idx[0], ng[0])[None, None, :]]
        if kfrac is not None:
            ph = [np.exp(2j * np.pi * kfrac[d] * np.floor_divide(idx[d], ng[d])) for d in range(3)]
            sub = sub * ph[2][None, :, None, None] * ph[1][None, None, :, None] * ph[0][None, None, None, :]
        t = np.einsum("bzyx,lx->bzyl", sub, tab[0])
        t = np.einsum("bzyl,my->bzml", t, tab[1])
        t = np.einsum("bzml,nz->bnml", t, tab[2])      # [b][nz][ny][nx]
        for nz in range(numax + 1):
            for ny in range(numax + 1 - nz):
                for nx in range(numax + 1 - nz - ny):
                    out[a, :, oracle.index(nx, ny, nz, numax)] = h ** 3 * t[:, nz, ny, nx]
    return out


# ----------------------------------------------------------------------------------------------
# P8: index set


def test_nsho_matches_values_printed_in_paper(golden):
    for numax, n in golden("nsho_paper.txt"):
        assert oracle.nsho(int(numax)) == int(n)
    # eq. (18) continues: 120 and 220 for numax 7 and 9 (used by BASELINE configs 3-5)
    assert oracle.nsho(7) == 8 * 9 * 10 // 6 == 120
    assert oracle.nsho(9) == 10 * 11 * 12 // 6 == 220


def test_index_is_a_bijection_with_paper_degeneracies(golden):
    deg = {int(nu): int(c) for nu, c in golden("degeneracy_paper.txt")}
    for numax in range(0, 10):
        seen = {}
        for nz in range(numax + 1):
            for ny in range(numax + 1 - nz):
                for nx in range(numax + 1 - nz - ny):
                    seen[oracle.index(nx, ny, nz, numax)] = (nx, ny, nz)
        assert sorted(seen) == list(range(oracle.nsho(numax)))
        for nu in range(numax + 1):
            assert sum(1 for t in seen.values() if sum(t) == nu) == deg[nu]
        assert oracle.index(numax + 1, 0, 0, numax) == -1
        assert oracle.index(-1, 0, 0, numax) == -1


def test_index_order_reading_A8():
    # nx fastest, then ny, then nz
    assert [oracle.index(*t, 1) for t in [(0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1)]] == [0, 1, 2, 3]
    order2 = [(0, 0, 0), (1, 0, 0), (2, 0, 0), (0, 1, 0), (1, 1, 0), (0, 2, 0), (0, 0, 1), (1, 0, 1), (0, 1, 1), (0, 0, 2)]
    assert [oracle.index(*t, 2) for t in order2] == list(range(10))


# ----------------------------------------------------------------------------------------------
# 1D functions


def test_hermite_matches_paper_recurrence_eq31(golden):
    xs = np.linspace(-6.0, 6.0, 49)
    for row in golden("hermite_recurrence_paper.txt"):
        n = int(row[0])
        coef = [float(c) for c in row[1:]]
        for x in xs:
            monic = sum(c * x ** k for k, c in enumerate(coef))
            got = oracle.hermite_phys(n, float(x))
            assert got == pytest.approx(2.0 ** n * monic, rel=1e-13, abs=1e-12)


def test_hermite_matches_scipy_library():
    rng = np.random.default_rng(1)
    for n in range(0, 16):
        for x in rng.uniform(-7, 7, size=40):
            ref = special.eval_hermite(n, x)
            scale = max(abs(ref), (2 * abs(x)) ** n, 1.0)
            assert abs(oracle.hermite_phys(n, float(x)) - ref) <= 5e-14 * scale


def test_phi_ground_state_value(golden):
    vals = {k: float(v) for k, v in golden("closed_forms.txt")}
    assert oracle.phi(0, 0.0, 1.0) == pytest.approx(vals["phi0_at_0_sigma1"], rel=1e-15)
    # width scaling: phi_n(u; sigma) = sigma^-1/2 phi_n(u/sigma; 1)
    assert oracle.phi(3, 0.7 * 1.3, 1.3) == pytest.approx(oracle.phi(3, 0.7, 1.0) / math.sqrt(1.3), rel=1e-14)


def test_phi_matches_scipy_and_parity():
    rng = np.random.default_rng(2)
    for sigma in (0.7, 1.0, 1.4):
        for n in range(0, 12):
            for u in rng.uniform(-6 * sigma, 6 * sigma, size=25):
                got = oracle.phi(n, float(u), sigma)
                assert abs(got - lib_phi(n, u, sigma)) <= 2e-14
                assert abs(oracle.phi(n, float(-u), sigma) - (-1) ** n * got) <= 1e-15


@pytest.mark.parametrize("sigma,h,numax", [(1.0, 0.25, 3), (0.8, 0.2, 5), (1.2, 0.2, 5), (1.0, 0.2, 7),
                                           (1.4, 0.15, 7), (0.7, 0.2, 9), (1.3, 0.2, 9)])
def test_P1_orthonormality_on_wide_grid(sigma, h, numax):
    """h sum_i phi_n(u_i) phi_m(u_i) = delta_nm on a wide cut (12 sigma), any grid offset.
    Holds to rounding because h < h_max = pi sigma / sqrt(2 numax + 1) (eq. 29)."""
    assert h < math.pi * sigma / math.sqrt(2 * numax + 1)
    for offset in (0.0, 0.37 * h, 0.5 * h):
        i = np.arange(-int(12 * sigma / h) - 1, int(12 * sigma / h) + 2)
        u = i * h - offset
        tab = np.array([[oracle.phi(n, float(x), sigma) for x in u] for n in range(numax + 1)])
        gram = h * tab @ tab.T
        assert np.max(np.abs(gram - np.eye(numax + 1))) < 5e-14


# ----------------------------------------------------------------------------------------------
# boxes (reading A3/A5), hand-computed


def test_box_ranges_hand_computed():
    # cfg 1: atom at 4.0, sigma 1, h 0.25, rc 6: (4-6)/0.25 = -8 exactly, (4+6)/0.25 = 40 exactly (inclusive)
    lo, hi, empty = oracle.box((32, 32, 32), 0.25, (1, 1, 1), (4.0, 4.0, 4.0), 1.0)
    assert list(lo) == [-8] * 3 and list(hi) == [40] * 3 and not empty
    lo, hi, empty = oracle.box((32, 32, 32), 0.25, (0, 0, 0), (4.0, 4.0, 4.0), 1.0)
    assert list(lo) == [0] * 3 and list(hi) == [31] * 3 and not empty
    # (0.05-6)/0.2 = -29.75 -> ceil -29 ; (0.05+6)/0.2 = 30.25 -> floor 30
    lo, hi, _ = oracle.box((96, 96, 96), 0.2, (1, 0, 1), (0.05, 0.05, 19.15), 1.0)
    assert (lo[0], hi[0]) == (-29, 30)
    assert (lo[1], hi[1]) == (0, 30)
    # (19.15-6)/0.2 = 65.75 -> 66 ; (19.15+6)/0.2 = 125.75 -> 125
    assert (lo[2], hi[2]) == (66, 125)
    # atom far outside an isolated grid: empty box
    _, _, empty = oracle.box((32, 32, 32), 0.25, (0, 0, 0), (4.0, 4.0, 30.0), 1.0)
    assert empty
    # narrower cut
    lo, hi, _ = oracle.box((64, 64, 64), 0.5, (1, 1, 1), (10.1, 10.1, 10.1), 0.5, 3.0)
    assert (lo[0], hi[0]) == (18, 23)      # 8.6/0.5 = 17.2 -> 18 ; 11.6/0.5 = 23.2 -> 23


# ----------------------------------------------------------------------------------------------
# P2: the literal triple sum equals the separable contraction (scipy tables, numpy einsum)


def test_P2_bruteforce_equals_separable_real_wrap():
    rng = np.random.default_rng(3)
    ng, h, per = (20, 18, 22), 0.3, (1, 1, 1)
    pos = np.array([[0.2, 5.1, 3.3], [5.9, 0.1, 6.5], [3.0, 2.7, 0.05]])
    sigma = np.array([0.35, 0.3, 0.4])
    psi = rng.standard_normal((2, ng[2], ng[1], ng[0]))
    got = oracle.project(ng, h, per, None, pos, sigma, 4, psi)
    ref = separable_project(ng, h, per, None, pos, sigma, 4, psi, 6.0)
    assert np.max(np.abs(got - ref)) < 1e-13 * np.max(np.abs(ref))


def test_P2_bruteforce_equals_separable_complex_bloch_and_isolated_axis():
    rng = np.random.default_rng(4)
    ng, h, per = (16, 24, 20), 0.25, (1, 0, 1)
    kfrac = (0.1, 0.0, 0.3)
    pos = np.array([[0.1, 0.4, 4.9], [3.9, 5.8, 0.2]])
    sigma = np.array([0.3, 0.28])
    psi = rng.standard_normal((2, ng[2], ng[1], ng[0])) + 1j * rng.standard_normal((2, ng[2], ng[1], ng[0]))
    got = oracle.project(ng, h, per, kfrac, pos, sigma, 3, psi)
    ref = separable_project(ng, h, per, kfrac, pos, sigma, 3, psi, 6.0)
    assert np.max(np.abs(got - ref)) < 1e-13 * np.max(np.abs(ref))


def test_full_3d_product_on_tiny_grid():
    """Brute force with the full 3D projector built by an outer product (numpy), one atom, no wrap."""
    rng = np.random.default_rng(5)
    ng, h = (14, 12, 10), 0.4
    pos, sigma, numax = np.array([[2.9, 2.3, 2.1]]), np.array([0.3]), 2
    psi = rng.standard_normal((1, ng[2], ng[1], ng[0]))
    got = oracle.project(ng, h, (0, 0, 0), None, pos, sigma, numax, psi)
    lo, hi = lib_ranges(ng, h, (0, 0, 0), pos[0], sigma[0], 6.0)
    x, y, z = (np.arange(ng[d]) * h - pos[0][d] for d in range(3))
    mask = [((np.arange(ng[d]) >= lo[d]) & (np.arange(ng[d]) <= hi[d])).astype(float) for d in range(3)]
    for nz in range(numax + 1):
        for ny in range(numax + 1 - nz):
            for nx in range(numax + 1 - nz - ny):
                P = np.einsum("z,y,x->zyx", lib_phi(nz, z, 0.3) * mask[2], lib_phi(ny, y, 0.3) * mask[1],
                              lib_phi(nx, x, 0.3) * mask[0])
                ref = h ** 3 * np.sum(P * psi[0])
                assert got[0, 0, oracle.index(nx, ny, nz, numax)] == pytest.approx(ref, rel=1e-12, abs=1e-15)


# ----------------------------------------------------------------------------------------------
# P3: Gaussian closed form


def gaussian_overlap_1d(n, sigma, s, d):
    """integral phi_n(x; sigma) exp(-(x-d)^2 / (2 s^2)) dx by scipy quadrature (library Hermite)."""
    f = lambda x: lib_phi(n, x, sigma) * math.exp(-0.5 * ((x - d) / s) ** 2)
    with warnings.catch_warnings():
        warnings.simplefilter("ignore", integrate.IntegrationWarning)   # tolerance is at rounding level
        val, _ = integrate.quad(f, -14 * sigma, 14 * sigma, epsabs=1e-14, epsrel=1e-13, limit=400)
    return val


def gaussian_overlap_closed(n, sigma, s, d):
    """SURVEY.md 8(c) P3 closed form; checked against quadrature in the test below."""
    S = sigma * sigma + s * s
    pref = sigma * s * math.sqrt(2 * math.pi / S) * math.exp(-d * d / (2 * S))
    norm = 1.0 / math.sqrt(2.0 ** n * math.factorial(n) * math.sqrt(math.pi) * sigma)
    tot = 0.0
    for k in range(n // 2 + 1):
        tot += ((-1) ** k * math.factorial(n) / (math.factorial(k) * math.factorial(n - 2 * k))
                * (2 * d * sigma / S) ** (n - 2 * k) * ((sigma * sigma - s * s) / S) ** k)
    return pref * norm * tot


def test_P3_closed_form_agrees_with_quadrature():
    for n in range(0, 8):
        for sigma, s, d in [(1.0, 1.0, 0.0), (0.9, 0.7, 0.3), (1.2, 1.5, -0.8)]:
            assert gaussian_overlap_closed(n, sigma, s, d) == pytest.approx(
                gaussian_overlap_1d(n, sigma, s, d), rel=1e-11, abs=1e-13)


def test_P3_gaussian_projection_c000(golden):
    vals = {k: float(v) for k, v in golden("closed_forms.txt")}
    ng, h, sigma, numax = (64, 64, 64), 0.25, 1.0, 3
    R = np.array([[8.0, 8.0, 8.0]])
    ax = [np.arange(ng[d]) * h - R[0][d] for d in range(3)]
    psi = np.exp(-0.5 * (ax[2][:, None, None] ** 2 + ax[1][None, :, None] ** 2 + ax[0][None, None, :] ** 2))[None]
    c = oracle.project(ng, h, (0, 0, 0), None, R, np.array([sigma]), numax, psi, rcut_sigma=7.5)
    assert c[0, 0, 0] == pytest.approx(vals["c000_gaussian_sigma1"], rel=2e-13)
    assert np.max(np.abs(c[0, 0, 1:])) < 1e-12


def test_P3_gaussian_projection_general():
    """Off-centre Gaussian of different width, distinct offsets per axis (catches axis transposition,
    a dropped h^3, a wrong normalisation)."""
    ng, h, sigma, s, numax = (80, 72, 88), 0.2, 0.8, 0.6, 4
    R = np.array([[8.03, 7.11, 8.86]])
    d = np.array([0.31, -0.22, 0.47])
    ax = [np.arange(ng[k]) * h - (R[0][k] + d[k]) for k in range(3)]
    psi = np.exp(-0.5 * (ax[2][:, None, None] ** 2 + ax[1][None, :, None] ** 2 + ax[0][None, None, :] ** 2) / s ** 2)[None]
    c = oracle.project(ng, h, (0, 0, 0), None, R, np.array([sigma]), numax, psi, rcut_sigma=8.5)
    one = [[gaussian_overlap_1d(n, sigma, s, d[k]) for n in range(numax + 1)] for k in range(3)]
    for nz in range(numax + 1):
        for ny in range(numax + 1 - nz):
            for nx in range(numax + 1 - nz - ny):
                ref = one[0][nx] * one[1][ny] * one[2][nz]
                assert c[0, 0, oracle.index(nx, ny, nz, numax)] == pytest.approx(ref, rel=1e-10, abs=2e-13)


# ----------------------------------------------------------------------------------------------
# P5: plane wave (Hermite functions are Fourier eigenfunctions, eq. (30))


def test_P5_plane_wave_with_wrap_and_bloch_phase():
    ng, h = (40, 36, 44), 0.25
    L = np.array(ng) * h
    kfrac = (0.1, 0.2, 0.3)
    m = np.array([1, -2, 3])
    q = 2 * np.pi * (m + np.array(kfrac)) / L
    x, y, z = (np.arange(ng[d]) * h for d in range(3))
    psi = np.exp(1j * (q[2] * z[:, None, None] + q[1] * y[None, :, None] + q[0] * x[None, None, :]))[None]
    pos = np.array([[0.3, 8.8, 5.2], [9.9, 0.1, 10.7]])
    sigma = np.array([0.5, 0.45])
    numax = 5
    # 11 sigma cut: box (44-45 points) is wider than the cell in x and y -> several images (reading A4)
    c = oracle.project(ng, h, (1, 1, 1), kfrac, pos, sigma, numax, psi, rcut_sigma=11.0)
    for a in range(2):
        f = [[math.sqrt(2 * math.pi * sigma[a]) * (1j ** n) * lib_phi(n, q[d] * sigma[a], 1.0)
              for n in range(numax + 1)] for d in range(3)]
        phase = np.exp(1j * np.dot(q, pos[a]))
        for nz in range(numax + 1):
            for ny in range(numax + 1 - nz):
                for nx in range(numax + 1 - nz - ny):
                    ref = phase * f[0][nx] * f[1][ny] * f[2][nz]
                    assert abs(c[a, 0, oracle.index(nx, ny, nz, numax)] - ref) < 1e-12


# ----------------------------------------------------------------------------------------------
# P4: adjoint identity <P psi, c> = h^3 <psi, A c>


@pytest.mark.parametrize("cplx", [False, True])
def test_P4_adjoint_identity(cplx):
    rng = np.random.default_rng(6)
    ng, h, per = (20, 24, 18), 0.3, (1, 1, 1)
    kfrac = (0.15, -0.2, 0.35) if cplx else None
    pos = rng.uniform(0, 1, size=(4, 3)) * np.array(ng) * h
    sigma = rng.uniform(0.3, 0.42, size=4)
    numax, nb = 3, 2
    shape = (nb, ng[2], ng[1], ng[0])
    psi = rng.standard_normal(shape) + (1j * rng.standard_normal(shape) if cplx else 0)
    cshape = (4, nb, oracle.nsho(numax))
    c = rng.standard_normal(cshape) + (1j * rng.standard_normal(cshape) if cplx else 0)
    Ppsi = oracle.project(ng, h, per, kfrac, pos, sigma, numax, psi)
    Ac = oracle.add(ng, h, per, kfrac, pos, sigma, numax, c, np.zeros_like(psi))
    lhs = np.sum(np.conj(Ppsi) * c)
    rhs = h ** 3 * np.sum(np.conj(psi) * Ac)
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)


def test_add_is_linear_and_accumulates():
    rng = np.random.default_rng(7)
    ng, h, per = (16, 16, 16), 0.3, (1, 1, 0)
    pos = rng.uniform(0, 1, size=(3, 3)) * np.array(ng) * h
    sigma = np.full(3, 0.35)
    c = rng.standard_normal((3, 1, oracle.nsho(2)))
    psi0 = rng.standard_normal((1, 16, 16, 16))
    a1 = oracle.add(ng, h, per, None, pos, sigma, 2, c, psi0)
    a0 = oracle.add(ng, h, per, None, pos, sigma, 2, c, np.zeros_like(psi0))
    assert np.max(np.abs(a1 - (psi0 + a0))) < 1e-14
    a2 = oracle.add(ng, h, per, None, pos, sigma, 2, 2.5 * c, np.zeros_like(psi0))
    assert np.max(np.abs(a2 - 2.5 * a0)) < 1e-13


@pytest.mark.parametrize("cplx", [False, True])
def test_add_points_matches_full_add(cplx):
    """The point-wise evaluation (used for sampled parity at full size) equals the box-loop add,
    including a box wider than the cell (several images per point)."""
    rng = np.random.default_rng(8)
    ng, h, per = (14, 16, 12), 0.3, (1, 1, 1)
    kfrac = (0.1, 0.2, 0.3) if cplx else None
    pos = rng.uniform(0, 1, size=(3, 3)) * np.array(ng) * h
    sigma = np.array([0.3, 0.38, 0.45])            # 12*0.45/0.3 = 18 points > 12..16: multi-image
    numax, nb = 3, 2
    cshape = (3, nb, oracle.nsho(numax))
    c = rng.standard_normal(cshape) + (1j * rng.standard_normal(cshape) if cplx else 0)
    full = oracle.add(ng, h, per, kfrac, pos, sigma, numax, c,
                      np.zeros((nb, ng[2], ng[1], ng[0]), dtype=c.dtype))
    pts = np.stack([rng.integers(0, ng[0], 200), rng.integers(0, ng[1], 200), rng.integers(0, ng[2], 200)], axis=1)
    bands = rng.integers(0, nb, 200)
    got = oracle.add_points(ng, h, per, kfrac, pos, sigma, numax, c, pts, bands)
    ref = full[bands, pts[:, 2], pts[:, 1], pts[:, 0]]
    assert np.max(np.abs(got - ref)) < 1e-13 * max(1.0, np.max(np.abs(ref)))


# ----------------------------------------------------------------------------------------------
# P6 / P7: invariances


def test_P6_lattice_translation_and_grid_roll():
    rng = np.random.default_rng(9)
    ng, h, per = (24, 20, 28), 0.25, (1, 1, 1)
    L = np.array(ng) * h
    pos = rng.uniform(0, 1, size=(3, 3)) * L
    sigma = np.array([0.3, 0.35, 0.4])
    psi = rng.standard_normal((2, ng[2], ng[1], ng[0]))
    c0 = oracle.project(ng, h, per, None, pos, sigma, 4, psi)
    # shift every atom by a lattice vector: same coefficients (real data)
    c1 = oracle.project(ng, h, per, None, pos + L * np.array([1, -1, 2]), sigma, 4, psi)
    assert np.max(np.abs(c1 - c0)) < 1e-12 * np.max(np.abs(c0))
    # shift atoms and psi together by whole grid points
    s = (3, -5, 7)
    psi_r = np.roll(psi, shift=(s[2], s[1], s[0]), axis=(1, 2, 3))
    c2 = oracle.project(ng, h, per, None, np.mod(pos + np.array(s) * h, L), sigma, 4, psi_r)
    assert np.max(np.abs(c2 - c0)) < 1e-12 * np.max(np.abs(c0))


def test_P6_bloch_phase_of_a_lattice_translation():
    rng = np.random.default_rng(10)
    ng, h, per, kfrac = (20, 20, 20), 0.25, (1, 1, 1), (0.1, 0.2, 0.3)
    L = np.array(ng) * h
    pos = rng.uniform(0, 1, size=(2, 3)) * L
    sigma = np.array([0.3, 0.33])
    shape = (1, 20, 20, 20)
    psi = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    c0 = oracle.project(ng, h, per, kfrac, pos, sigma, 3, psi)
    mvec = np.array([1, 0, -1])
    c1 = oracle.project(ng, h, per, kfrac, pos + L * mvec, sigma, 3, psi)
    # psi(r + L m) = exp(2 pi i kfrac.m) psi(r)  (reading A6)
    assert np.max(np.abs(c1 - np.exp(2j * np.pi * np.dot(kfrac, mvec)) * c0)) < 1e-12 * np.max(np.abs(c0))


def test_P7_isolated_equals_periodic_on_zero_padded_grid():
    rng = np.random.default_rng(11)
    ng, h = (16, 14, 18), 0.3
    pos = np.array([[0.4, 2.0, 5.1], [4.5, 4.0, 0.2]])
    sigma = np.array([0.3, 0.36])
    psi = rng.standard_normal((1, ng[2], ng[1], ng[0]))
    c_iso = oracle.project(ng, h, (0, 0, 0), None, pos, sigma, 3, psi)
    pad = 16
    big = tuple(n + 2 * pad for n in ng)
    psi_big = np.zeros((1, big[2], big[1], big[0]))
    psi_big[:, pad:pad + ng[2], pad:pad + ng[1], pad:pad + ng[0]] = psi
    c_per = oracle.project(big, h, (1, 1, 1), None, pos + pad * h, sigma, 3, psi_big)
    assert np.max(np.abs(c_iso - c_per)) < 1e-13 * np.max(np.abs(c_iso))
    # add: isolated add equals the interior of the padded periodic add
    c = rng.standard_normal((2, 1, oracle.nsho(3)))
    a_iso = oracle.add(ng, h, (0, 0, 0), None, pos, sigma, 3, c, np.zeros_like(psi))
    a_per = oracle.add(big, h, (1, 1, 1), None, pos + pad * h, sigma, 3, c, np.zeros_like(psi_big))
    inner = a_per[:, pad:pad + ng[2], pad:pad + ng[1], pad:pad + ng[0]]
    assert np.max(np.abs(a_iso - inner)) < 1e-13 * np.max(np.abs(a_iso))


def test_complex_projection_is_linear_in_re_im_parts():
    rng = np.random.default_rng(12)
    ng, h, per = (16, 16, 16), 0.3, (1, 1, 1)
    pos = rng.uniform(0, 1, size=(2, 3)) * 4.8
    sigma = np.array([0.3, 0.36])
    re = rng.standard_normal((1, 16, 16, 16))
    im = rng.standard_normal((1, 16, 16, 16))
    cz = oracle.project(ng, h, per, (0.0, 0.0, 0.0), pos, sigma, 3, re + 1j * im)
    cr = oracle.project(ng, h, per, None, pos, sigma, 3, re)
    ci = oracle.project(ng, h, per, None, pos, sigma, 3, im)
    assert np.max(np.abs(cz - (cr + 1j * ci))) < 1e-14


def test_degenerate_cases():
    # atom entirely outside an isolated grid: zero coefficients, add is a no-op
    ng, h = (8, 8, 8), 0.5
    pos, sigma = np.array([[2.0, 2.0, 40.0]]), np.array([0.5])
    psi = np.ones((1, 8, 8, 8))
    c = oracle.project(ng, h, (0, 0, 0), None, pos, sigma, 2, psi)
    assert np.all(c == 0.0)
    out = oracle.add(ng, h, (0, 0, 0), None, pos, sigma, 2, np.ones((1, 1, oracle.nsho(2))), psi)
    assert np.array_equal(out, psi)
    # no atoms at all
    c = oracle.project(ng, h, (1, 1, 1), None, np.zeros((0, 3)), np.zeros(0), 2, psi)
    assert c.shape == (0, 1, 10)
    # numax = 0: a single Gaussian per atom
    # projection of the constant 1 onto phi_0^3D: (integral phi_0)^3 = (sqrt(2) pi^(1/4) sigma^(1/2))^3;
    # the 8 sigma box (26 points) is wider than the 16-point cell: every image counts once (reading A4)
    c = oracle.project((16, 16, 16), 0.25, (1, 1, 1), None, np.array([[2.0, 2.1, 1.9]]), np.array([0.4]), 0,
                       np.ones((1, 16, 16, 16)), rcut_sigma=8.0)
    assert c[0, 0, 0] == pytest.approx((math.sqrt(2) * math.pi ** 0.25 * math.sqrt(0.4)) ** 3, rel=1e-12)


# ----------------------------------------------------------------------------------------------
# the explicit-pair branch of oracle_project_pairs (pair_atom / pair_band lists, bands in separate
# buffers through psi_band_ptrs): every full-size GPU parity check rests on it


def test_project_pairs_explicit_branch_gaussian_closed_form():
    """P3 through the explicit-pair branch: two atoms, three bands held in SEPARATE buffers, a shuffled pair
    list with a repeated pair; band 1 is an off-centre Gaussian around atom 1 whose coefficients have the
    closed form of test_P3_gaussian_projection_general, band 2 one around atom 0 (transposed atom / band
    indices, a wrong output row or a wrong band pointer all fail)."""
    ng, h, numax = (72, 80, 64), 0.2, 4
    sigma = np.array([0.8, 0.7])
    R = np.array([[7.13, 8.02, 6.31], [7.49, 7.77, 6.58]])
    s = [None, 0.6, 0.75]
    d = [None, np.array([0.21, -0.32, 0.17]), np.array([-0.25, 0.14, 0.33])]
    centre = [None, R[1] + d[1], R[0] + d[2]]
    rng = np.random.default_rng(21)
    bands = {0: rng.standard_normal((ng[2], ng[1], ng[0]))}
    for b in (1, 2):
        ax = [np.arange(ng[k]) * h - centre[b][k] for k in range(3)]
        bands[b] = np.exp(-0.5 * (ax[2][:, None, None] ** 2 + ax[1][None, :, None] ** 2 + ax[0][None, None, :] ** 2) / s[b] ** 2)
    pa = np.array([1, 0, 1, 0, 1])
    pb = np.array([1, 2, 0, 0, 1])
    c = oracle.project_pairs(ng, h, (0, 0, 0), None, R, sigma, numax, bands, pa, pb, 3, False, rcut_sigma=8.5)
    assert c.shape == (5, oracle.nsho(numax))
    for row, (a, b) in ((0, (1, 1)), (1, (0, 2)), (4, (1, 1))):
        one = [[gaussian_overlap_1d(n, sigma[a], s[b], d[b][k]) for n in range(numax + 1)] for k in range(3)]
        for nz in range(numax + 1):
            for ny in range(numax + 1 - nz):
                for nx in range(numax + 1 - nz - ny):
                    ref = one[0][nx] * one[1][ny] * one[2][nz]
                    assert c[row, oracle.index(nx, ny, nz, numax)] == pytest.approx(ref, rel=1e-10, abs=2e-13)
    assert np.array_equal(c[0], c[4])


@pytest.mark.parametrize("cplx", [False, True])
def test_project_pairs_explicit_branch_equals_rows_of_full_projection(cplx):
    """A shuffled subset of (atom, band) pairs, bands passed as separate buffers, equals the matching rows
    of the full projection (wrap, Bloch phase) and of the separable numpy contraction with scipy tables."""
    rng = np.random.default_rng(22)
    ng, h, per = (18, 22, 20), 0.3, (1, 1, 1)
    kfrac = (0.1, 0.2, 0.3) if cplx else None
    pos = rng.uniform(0, 1, size=(5, 3)) * np.array(ng) * h
    sigma = rng.uniform(0.3, 0.4, size=5)
    numax, nb = 3, 4
    shape = (nb, ng[2], ng[1], ng[0])
    psi = rng.standard_normal(shape) + (1j * rng.standard_normal(shape) if cplx else 0)
    full = oracle.project(ng, h, per, kfrac, pos, sigma, numax, psi, rcut_sigma=5.0)
    sep = separable_project(ng, h, per, kfrac, pos, sigma, numax, psi, 5.0)
    pairs = [(a, b) for a in range(5) for b in range(nb)]
    sel = rng.permutation(len(pairs))[:11]
    pa = np.array([pairs[i][0] for i in sel])
    pb = np.array([pairs[i][1] for i in sel])
    bands = {int(b): psi[int(b)].copy() for b in np.unique(pb)}      # separate buffers, only the bands in use
    got = oracle.project_pairs(ng, h, per, kfrac, pos, sigma, numax, bands, pa, pb, nb, cplx, rcut_sigma=5.0)
    assert np.array_equal(got, full[pa, pb])
    assert np.max(np.abs(got - sep[pa, pb])) < 1e-13 * np.max(np.abs(sep))


@pytest.mark.parametrize("cplx", [False, True])
def test_add_points_bands_matches_full_add(cplx):
    """The all-bands point-wise evaluation equals the box-loop add (multi-image boxes, Bloch phase, an
    isolated axis) for a subset of bands given in a shuffled order."""
    rng = np.random.default_rng(23)
    ng, h, per = (14, 16, 12), 0.3, (1, 1, 0)
    kfrac = (0.1, 0.2, 0.0) if cplx else None
    pos = rng.uniform(0, 1, size=(3, 3)) * np.array(ng) * h
    sigma = np.array([0.3, 0.38, 0.45])
    numax, nb = 3, 5
    cshape = (3, nb, oracle.nsho(numax))
    c = rng.standard_normal(cshape) + (1j * rng.standard_normal(cshape) if cplx else 0)
    full = oracle.add(ng, h, per, kfrac, pos, sigma, numax, c, np.zeros((nb, ng[2], ng[1], ng[0]), dtype=c.dtype))
    pts = np.stack([rng.integers(0, ng[0], 150), rng.integers(0, ng[1], 150), rng.integers(0, ng[2], 150)], axis=1)
    sel = np.array([4, 0, 2])
    got = oracle.add_points_bands(ng, h, per, kfrac, pos, sigma, numax, c, pts, sel)
    ref = full[sel][:, pts[:, 2], pts[:, 1], pts[:, 0]].T
    assert got.shape == (150, 3)
    assert np.max(np.abs(got - ref)) < 1e-13 * max(1.0, np.max(np.abs(ref)))


# ----------------------------------------------------------------------------------------------
# step (2): d = D c  (eq. (27)-(28) PAPER.md:252-262)


def test_dmul_hand_written_2x2_and_identity():
    # d_i = sum_j D_ij c_j with D = [[2, -1], [3, 0.5]] (NOT symmetric: a transposed D fails), two bands
    D = np.array([[[2.0, -1.0], [3.0, 0.5]]])
    c = np.array([[[1.0, 4.0], [-2.0, 0.25]]])
    d = oracle.dmul(D, c)
    assert np.array_equal(d, np.array([[[2.0 * 1 - 1.0 * 4, 3.0 * 1 + 0.5 * 4], [2.0 * -2 - 0.25, 3.0 * -2 + 0.125]]]))
    cz = c + 1j * np.array([[[0.5, -1.0], [2.0, 8.0]]])
    dz = oracle.dmul(D, cz)
    assert np.array_equal(dz.real, d)
    assert np.array_equal(dz.imag, np.array([[[2.0 * 0.5 + 1.0, 3.0 * 0.5 - 0.5], [2.0 * 2 - 8.0, 3.0 * 2 + 4.0]]]))
    rng = np.random.default_rng(24)
    c = rng.standard_normal((3, 2, 10))
    assert np.array_equal(oracle.dmul(np.tile(np.eye(10), (3, 1, 1)), c), c)


@pytest.mark.parametrize("cplx", [False, True])
def test_dmul_matches_library_matmul_per_atom(cplx):
    rng = np.random.default_rng(25)
    na, nb, n = 4, 3, oracle.nsho(3)
    D = rng.standard_normal((na, n, n))
    c = rng.standard_normal((na, nb, n)) + (1j * rng.standard_normal((na, nb, n)) if cplx else 0)
    ref = np.einsum("aij,abj->abi", D, c)
    assert np.max(np.abs(oracle.dmul(D, c) - ref)) < 1e-13 * np.max(np.abs(ref))


@pytest.mark.parametrize("cplx", [False, True])
def test_nonlocal_action_is_hermitian_for_symmetric_D(cplx):
    """V = A D P (steps (1)-(3)) with real symmetric D per atom is Hermitian:
    <phi, V psi> = conj(<psi, V phi>) (grid inner product; add = P^H / h^3, reading A7).  With D = 1 the
    action reduces to add(project(psi))."""
    rng = np.random.default_rng(26)
    ng, h, per = (18, 16, 20), 0.3, (1, 1, 1)
    kfrac = (0.15, -0.2, 0.35) if cplx else None
    pos = rng.uniform(0, 1, size=(3, 3)) * np.array(ng) * h
    sigma = rng.uniform(0.3, 0.4, size=3)
    numax = 3
    n = oracle.nsho(numax)
    D = rng.standard_normal((3, n, n))
    D = D + np.transpose(D, (0, 2, 1))
    shape = (1, ng[2], ng[1], ng[0])
    psi = rng.standard_normal(shape) + (1j * rng.standard_normal(shape) if cplx else 0)
    phi = rng.standard_normal(shape) + (1j * rng.standard_normal(shape) if cplx else 0)

    def V(f, Dm):
        c = oracle.project(ng, h, per, kfrac, pos, sigma, numax, f, rcut_sigma=5.0)
        return oracle.add(ng, h, per, kfrac, pos, sigma, numax, oracle.dmul(Dm, c), np.zeros_like(f), rcut_sigma=5.0)

    lhs = np.sum(np.conj(phi) * V(psi, D))
    rhs = np.conj(np.sum(np.conj(psi) * V(phi, D)))
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)
    one = np.tile(np.eye(n), (3, 1, 1))
    c = oracle.project(ng, h, per, kfrac, pos, sigma, numax, psi, rcut_sigma=5.0)
    ref = oracle.add(ng, h, per, kfrac, pos, sigma, numax, c, np.zeros_like(psi), rcut_sigma=5.0)
    assert np.array_equal(V(psi, one), ref)


# ----------------------------------------------------------------------------------------------
# f4: the unitary transform U between Cartesian and spherical states (eq. (10)-(11))


def test_umatrix_textbook_shells(golden):
    """s, p, d and s* rows against the values every text lists (tests/golden/umatrix_textbook.txt); everything else
    inside the shells nu <= 2 must vanish."""
    U = oracle.umatrix(2)
    want = np.zeros_like(U)
    for nr, l, m, nx, ny, nz, v in golden("umatrix_textbook.txt"):
        want[oracle.rlm_index(int(nr), int(l), int(m), 2), oracle.index(int(nx), int(ny), int(nz), 2)] = float(v)
    assert np.max(np.abs(U - want)) < 1e-14
    # the same shells are the leading block of a larger basis in the spherical order, and the Cartesian columns agree
    U5 = oracle.umatrix(5)
    for nr, l, m, nx, ny, nz, v in golden("umatrix_textbook.txt"):
        assert U5[oracle.rlm_index(int(nr), int(l), int(m), 5), oracle.index(int(nx), int(ny), int(nz), 5)] == pytest.approx(float(v), abs=1e-14)


def test_umatrix_f_shell_rows_from_harmonic_polynomials(golden):
    """The whole f shell (l = 3, every m), the p* states and three g states against values that follow from the
    mathematics alone (tests/golden/umatrix_harmonic_polynomials.txt: integer coefficients of the textbook solid
    harmonics; U = p sqrt(a! b! c!) / norm).  An l-dependent sign slip or a wrong m order in the oracle's real
    spherical harmonics -- which orthogonality and the block structure would not notice -- fails here: f_xyz must be
    exactly the state |1 1 1>."""
    import math
    numax = 4
    U = oracle.umatrix(numax)
    rows = {}
    for nr, l, m, a, b, c, p in golden("umatrix_harmonic_polynomials.txt"):
        key = (int(nr), int(l), int(m))
        abc = (int(a), int(b), int(c))
        assert sum(abc) == key[1] + 2 * key[0]                                      # eq. (11): same shell
        rows.setdefault(key, {})[abc] = int(p) * math.sqrt(math.factorial(abc[0]) * math.factorial(abc[1]) * math.factorial(abc[2]))
    assert {k for k in rows if k[1] == 3} == {(0, 3, m) for m in range(-3, 4)}
    for (nr, l, m), wts in rows.items():
        norm = math.sqrt(sum(v * v for v in wts.values()))
        want = np.zeros(U.shape[1])
        for abc, v in wts.items():
            want[oracle.index(*abc, numax)] = v / norm
        got = U[oracle.rlm_index(nr, l, m, numax)]
        assert np.max(np.abs(got - want)) < 1e-14, (nr, l, m)
    assert U[oracle.rlm_index(0, 3, -2, numax), oracle.index(1, 1, 1, numax)] == pytest.approx(1.0, abs=1e-14)


@pytest.mark.parametrize("numax", [0, 1, 3, 6])
def test_umatrix_is_orthogonal_and_block_diagonal_in_nu(numax):
    """Unitarity ("a unitary transform") and eq. (11): elements vanish unless l + 2 nr = nx + ny + nz."""
    U = oracle.umatrix(numax)
    n = oracle.nsho(numax)
    assert U.shape == (n, n)
    assert np.max(np.abs(U @ U.T - np.eye(n))) < 1e-13 and np.max(np.abs(U.T @ U - np.eye(n))) < 1e-13
    nu_row = np.zeros(n, int)
    seen = set()
    for nu in range(numax + 1):
        for nr in range(nu // 2 + 1):
            l = nu - 2 * nr
            for m in range(-l, l + 1):
                i = oracle.rlm_index(nr, l, m, numax)
                assert 0 <= i < n and i not in seen
                seen.add(i)
                nu_row[i] = nu
    assert len(seen) == n                                                   # the spherical index is a bijection too
    for nz in range(numax + 1):
        for ny in range(numax + 1 - nz):
            for nx in range(numax + 1 - nz - ny):
                col = U[:, oracle.index(nx, ny, nz, numax)]
                assert np.max(np.abs(col[nu_row != nx + ny + nz]), initial=0.0) < 1e-14


def test_umatrix_rotates_a_spherically_symmetric_function_into_l0_only():
    """A property that does not use the matrix's own construction: psi(r) = exp(-r^2 / (2 s^2)) is spherically symmetric,
    so its Cartesian projection coefficients (closed form of pin P3, a product of 1D overlaps) must map under U onto the
    l = 0 states only."""
    numax, sigma, s = 6, 1.0, 0.8
    one = [gaussian_overlap_closed(n, sigma, s, 0.0) for n in range(numax + 1)]
    c = np.zeros(oracle.nsho(numax))
    for nz in range(numax + 1):
        for ny in range(numax + 1 - nz):
            for nx in range(numax + 1 - nz - ny):
                c[oracle.index(nx, ny, nz, numax)] = one[nx] * one[ny] * one[nz]
    d = oracle.umatrix(numax) @ c
    for nu in range(numax + 1):
        for nr in range(nu // 2 + 1):
            l = nu - 2 * nr
            for m in range(-l, l + 1):
                v = d[oracle.rlm_index(nr, l, m, numax)]
                if l > 0:
                    assert abs(v) < 1e-13
    assert abs(d[oracle.rlm_index(0, 0, 0, numax)]) > 1.0                   # and the s states carry it
    assert abs(np.sum(d * d) - np.sum(c * c)) < 1e-13
