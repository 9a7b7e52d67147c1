"""Oracle for the unitary transform U between the Cartesian and the spherical eigenstates of the 3D harmonic
oscillator (eq. (10)-(11)) -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see sho_oracle.c).

The paper states that U exists, that U[(nr,l,m)][(nx,ny,nz)] vanishes unless l + 2 nr = nu = nx + ny + nz (eq. (11))
and gives no formula for its elements.  The oracle takes the DEFINITION -- the overlap integral of the two families,
eq. (10) projected on one spherical state --

    U[(nr,l,m)][(nx,ny,nz)] = integral Psi_{nr l m}(r) Psi_{nx ny nz}(r) d^3r                     (sigma = 1)

with   Psi_{nx ny nz} = phi_nx(x) phi_ny(y) phi_nz(z)            eq. (4); phi_n orthonormal (reading A1)
       Psi_{nr l m}   = R_{nr l}(r) Y_lm(theta, phi)             eq. (7)
       R_{nr l}(r)    = N r^l L_nr^(l+1/2)(r^2) exp(-r^2/2)      eq. (8), N = sqrt(2 nr! / Gamma(nr + l + 3/2))

and evaluates it with a tensor Gauss-Hermite rule, which is EXACT here (the integrand is exp(-r^2) times a polynomial of
degree <= 2 numax per axis; numax + 1 nodes per axis suffice, numax + 3 are used).

Readings where the paper is silent (A17-A19):
  A17  order of the spherical index: nu ascending; inside a shell nr = 0, 1, ... (l = nu - 2 nr descending); m = -l .. l
  A18  Y_lm are the REAL spherical harmonics: Y_l0 = Y_l^0, Y_l,+m = sqrt(2) (-1)^m Re Y_l^m, Y_l,-m = sqrt(2) (-1)^m Im Y_l^m
       (Y_l^m with the Condon-Shortley phase), so Y_1,-1 ~ y, Y_10 ~ z, Y_11 ~ x with positive factors
  A19  signs: phi_n has a positive leading coefficient, R_{nr l} is positive for r -> 0 (L_n^(a)(0) > 0)
With these U is a real orthogonal matrix, and the coefficients in the spherical representation are c_rlm = U c_cart.
"""
from __future__ import annotations

import math

import numpy as np
from scipy import special

from .sho_oracle import index as cart_index
from .sho_oracle import nsho, phi


def rlm_index(nr: int, l: int, m: int, numax: int) -> int:
    """Position of (nr, l, m) in the spherical order of reading A17, by literal enumeration; -1 if not in the basis."""
    n = 0
    for nu in range(numax + 1):
        for r in range(nu // 2 + 1):
            ll = nu - 2 * r
            for mm in range(-ll, ll + 1):
                if (r, ll, mm) == (nr, l, m):
                    return n
                n += 1
    return -1


def real_sph_harm(l: int, m: int, theta, phi_):
    """Reading A18; theta polar, phi_ azimuth."""
    ma = abs(m)
    if hasattr(special, "sph_harm_y"):
        y = special.sph_harm_y(l, ma, theta, phi_)
    else:  # older scipy: sph_harm(m, l, azimuth, polar)
        y = special.sph_harm(ma, l, phi_, theta)
    if m == 0:
        return y.real
    s = math.sqrt(2.0) * (-1.0) ** ma
    return s * (y.real if m > 0 else y.imag)


def radial(nr: int, l: int, r):
    """Normalised R_{nr l}(r) of eq. (8), sigma = 1: integral R^2 r^2 dr = 1."""
    norm = math.sqrt(2.0 * math.factorial(nr) / special.gamma(nr + l + 1.5))
    return norm * r ** l * special.eval_genlaguerre(nr, l + 0.5, r * r) * np.exp(-0.5 * r * r)


def umatrix(numax: int) -> np.ndarray:
    """U[rlm_index][cart_index] (reading A17 rows, reading A8 columns), shape [N_SHO][N_SHO]."""
    n = nsho(numax)
    nq = numax + 3
    xq, wq = np.polynomial.hermite.hermgauss(nq)           # weight exp(-x^2)
    X, Y, Z = np.meshgrid(xq, xq, xq, indexing="ij")
    W = wq[:, None, None] * wq[None, :, None] * wq[None, None, :] * np.exp(X * X + Y * Y + Z * Z)   # plain dV weights
    R = np.sqrt(X * X + Y * Y + Z * Z)
    TH = np.arccos(np.clip(Z / np.maximum(R, 1e-300), -1.0, 1.0))
    PH = np.arctan2(Y, X)
    f1 = np.array([[phi(k, float(x), 1.0) for x in xq] for k in range(numax + 1)])       # [n][node]
    U = np.zeros((n, n))
    for nu in range(numax + 1):
        for nr in range(nu // 2 + 1):
            l = nu - 2 * nr
            for m in range(-l, l + 1):
                sph = radial(nr, l, R) * real_sph_harm(l, m, TH, PH) * W
                i = rlm_index(nr, l, m, numax)
                for nz in range(numax + 1):
                    for ny in range(numax + 1 - nz):
                        for nx in range(numax + 1 - nz - ny):
                            cart = f1[nx][:, None, None] * f1[ny][None, :, None] * f1[nz][None, None, :]
                            U[i, cart_index(nx, ny, nz, numax)] = float(np.sum(sph * cart))
    return U
