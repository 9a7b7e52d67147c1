// sho_umat.cu -- host code: the unitary transform U between the Cartesian SHO states (nx,ny,nz) and the spherical ones
// (nr,l,m), eq. (10)-(11) (f4).  The paper gives no formula for the elements; they are the overlap
// integrals  U[(nr,l,m)][(nx,ny,nz)] = integral Psi_{nr l m} Psi_{nx ny nz} d^3r  (sigma = 1), evaluated here exactly:
// both families are exp(-r^2/2) times a polynomial, so a tensor Gauss-Hermite rule with numax + 2 nodes per axis
// integrates their product without error beyond rounding.  Only pairs inside one shell nu = l + 2 nr = nx + ny + nz are
// computed (eq. (11)); the rest of the matrix is exact zeros.
//   polynomial part of Psi_{nx ny nz}: h_nx(x) h_ny(y) h_nz(z), h_{n+1} = sqrt(2/(n+1)) x h_n - sqrt(n/(n+1)) h_{n-1},
//       h_0 = pi^(-1/4)  (the orthonormal form of the recurrence of eq. (31))
//   polynomial part of Psi_{nr l m}:  N L_nr^(l+1/2)(r^2) S_lm(x,y,z), N = sqrt(2 nr! / Gamma(nr + l + 3/2)) (eq. (8),
//       PAPER.md:100), S_lm = r^l Y_lm the REAL solid harmonics built from the Cartesian recurrences
//       (x + i y)^m = A_m + i B_m and Q_l^m(z, r^2) = r^(l-m) d^m P_l / dt^m at t = z / r
// Conventions (readings A17-A19): rows ordered nu ascending, nr ascending inside a shell, m = -l..l; real
// harmonics with positive factors (S_1,-1 ~ y, S_10 ~ z, S_11 ~ x); R positive at the origin.  Shares nothing with oracle/.
#include <cmath>
#include <vector>

#include "sho_internal.h"

namespace {

const double kPi = 3.14159265358979323846264338327950288;

// nodes and weights of the n-point Gauss-Hermite rule (weight exp(-x^2)), Golub-Welsch style: the nodes are the
// eigenvalues of the Jacobi matrix of the Hermite recurrence (symmetric tridiagonal, zero diagonal, off-diagonal
// b_k = sqrt(k / 2), k = 1 .. n-1).  Eigenvalue i is bracketed by bisection on the Sturm count (number of eigenvalues
// below lambda = number of negative pivots of T - lambda I), then polished with Newton steps on the orthonormal
// polynomial p_n; the weight is the Christoffel number 1 / sum_{k<n} p_k(x_i)^2.  Roots in descending order.
void gauss_hermite(int n, std::vector<double>& x, std::vector<double>& w)
{
    x.assign(n, 0.0); w.assign(n, 0.0);
    auto below = [n](double lam) {                           // eigenvalues of the Jacobi matrix smaller than lam
        int count = 0;
        double q = -lam;
        for (int k = 1; k <= n; ++k) {
            if (q < 0.0) ++count;
            if (k == n) break;
            if (q == 0.0) q = 1e-300;
            q = -lam - 0.5 * k / q;
        }
        return count;
    };
    const double bound = std::sqrt(2.0 * n) + 1.0;           // Gershgorin: |x| <= 2 max b_k
    for (int i = 0; i < (n + 1) / 2; ++i) {                  // the i-th largest root; the rule is symmetric
        const int rank = n - 1 - i;                          // ascending position of that root
        double lo = -bound, hi = bound;
        for (int it = 0; it < 80; ++it) {
            const double mid = 0.5 * (lo + hi);
            if (below(mid) > rank) hi = mid; else lo = mid;
        }
        double z = (n % 2 == 1 && i == n / 2) ? 0.0 : 0.5 * (lo + hi);
        double sum = 0.0;
        for (int it = 0; it < 3; ++it) {
            double pm = 0.0, pc = std::pow(kPi, -0.25);      // p_0 .. p_n at z (orthonormal for the weight exp(-x^2))
            sum = 0.0;
            for (int k = 0; k < n; ++k) {
                sum += pc * pc;
                const double pn = z * std::sqrt(2.0 / (k + 1.0)) * pc - std::sqrt((double)k / (k + 1.0)) * pm;
                pm = pc; pc = pn;
            }
            if (z == 0.0) break;
            z -= pc / (std::sqrt(2.0 * n) * pm);             // p_n' = sqrt(2 n) p_{n-1}
        }
        x[i] = z; x[n - 1 - i] = -z;
        w[i] = 1.0 / sum; w[n - 1 - i] = w[i];
    }
}

double factorial_d(int n) { double f = 1.0; for (int i = 2; i <= n; ++i) f *= i; return f; }

}  // namespace

extern "C" int sho_rlm_index(int nr, int l, int m, int numax)
{
    if (numax < 0 || numax > SHO_NUMAX_MAX || nr < 0 || l < 0 || m < -l || m > l || l + 2 * nr > numax) return -1;
    const int nu = l + 2 * nr;
    int n = nu * (nu + 1) * (nu + 2) / 6;                 // states of the shells below nu
    for (int r = 0; r < nr; ++r) n += 2 * (nu - 2 * r) + 1;
    return n + (m + l);
}

extern "C" sho_status sho_umatrix(int numax, double* u)
{
    if (numax < 0 || numax > SHO_NUMAX_MAX || !u) { sho::set_error("sho_umatrix: bad argument"); return SHO_ERR_INVALID_ARG; }
    const int n = sho_nsho(numax);
    for (size_t i = 0; i < (size_t)n * n; ++i) u[i] = 0.0;
    const int nq = numax + 2;
    std::vector<double> xq, wq;
    gauss_hermite(nq, xq, wq);
    // h_k at the nodes
    std::vector<double> h((size_t)(numax + 1) * nq);
    for (int i = 0; i < nq; ++i) {
        double hm = 0.0, hc = std::pow(kPi, -0.25);
        for (int k = 0; k <= numax; ++k) {
            h[(size_t)k * nq + i] = hc;
            const double hn = std::sqrt(2.0 / (k + 1.0)) * xq[i] * hc - std::sqrt((double)k / (k + 1.0)) * hm;
            hm = hc; hc = hn;
        }
    }
    const int L = numax;
    std::vector<double> sph((size_t)n);                   // polynomial parts of all spherical states at one node
    std::vector<double> A(L + 1), B(L + 1), Q((size_t)(L + 1) * (L + 1));
    for (int ix = 0; ix < nq; ++ix)
        for (int iy = 0; iy < nq; ++iy)
            for (int iz = 0; iz < nq; ++iz) {
                const double x = xq[ix], y = xq[iy], z = xq[iz], r2 = x * x + y * y + z * z;
                const double wgt = wq[ix] * wq[iy] * wq[iz];
                A[0] = 1.0; B[0] = 0.0;
                for (int m = 1; m <= L; ++m) { A[m] = x * A[m - 1] - y * B[m - 1]; B[m] = x * B[m - 1] + y * A[m - 1]; }
                for (int m = 0; m <= L; ++m) {
                    double qmm = 1.0;
                    for (int k = 1; k <= m; ++k) qmm *= (2.0 * k - 1.0);                     // (2m-1)!!
                    Q[(size_t)m * (L + 1) + m] = qmm;
                    if (m + 1 <= L) Q[(size_t)(m + 1) * (L + 1) + m] = (2.0 * m + 1.0) * z * qmm;
                    for (int l = m + 2; l <= L; ++l)
                        Q[(size_t)l * (L + 1) + m] = ((2.0 * l - 1.0) * z * Q[(size_t)(l - 1) * (L + 1) + m] -
                                                      (l + m - 1.0) * r2 * Q[(size_t)(l - 2) * (L + 1) + m]) / (double)(l - m);
                }
                for (int nu = 0; nu <= numax; ++nu)
                    for (int nr = 0; 2 * nr <= nu; ++nr) {
                        const int l = nu - 2 * nr;
                        const double al = l + 0.5;
                        double lm1 = 0.0, lc = 1.0;                                          // Laguerre L_k^(al)(r2)
                        for (int k = 0; k < nr; ++k) {
                            const double ln = ((2.0 * k + 1.0 + al - r2) * lc - (k + al) * lm1) / (k + 1.0);
                            lm1 = lc; lc = ln;
                        }
                        const double rad = std::sqrt(2.0 * factorial_d(nr) / std::tgamma(nr + l + 1.5)) * lc;
                        for (int m = -l; m <= l; ++m) {
                            const int ma = m < 0 ? -m : m;
                            const double nlm = std::sqrt((2.0 * l + 1.0) / (4.0 * kPi) * factorial_d(l - ma) / factorial_d(l + ma));
                            const double ang = Q[(size_t)l * (L + 1) + ma] * (m == 0 ? 1.0 : std::sqrt(2.0) * (m > 0 ? A[ma] : B[ma]));
                            sph[(size_t)sho_rlm_index(nr, l, m, numax)] = rad * nlm * ang;
                        }
                    }
                for (int nz = 0; nz <= numax; ++nz)
                    for (int ny = 0; ny <= numax - nz; ++ny)
                        for (int nx = 0; nx <= numax - nz - ny; ++nx) {
                            const int nu = nx + ny + nz;
                            const double c = wgt * h[(size_t)nx * nq + ix] * h[(size_t)ny * nq + iy] * h[(size_t)nz * nq + iz];
                            const int j = sho_index(nx, ny, nz, numax);
                            const int i0 = nu * (nu + 1) * (nu + 2) / 6, i1 = (nu + 1) * (nu + 2) * (nu + 3) / 6;
                            for (int i = i0; i < i1; ++i) u[(size_t)i * n + j] += sph[(size_t)i] * c;
                        }
            }
    return SHO_OK;
}
