// lsms_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU oracle for the LSMS hot path
//     tau^{00} = [ (t^{-1} - g0)^{-1} ]_{00}                (eq. (4); :62)
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may load this file.  It shares no code with paper_2308_16317_b200/ (the CUDA
// path) and neither includes the other.  Plain C++17, std::complex, no BLAS/LAPACK,
// no blocking, no fusion: every routine is the textbook definition written out.
//
// The paper names the objects ("t is the single site scattering matrix
// and g0 is the free particle propagator between two different atom sites") but prints
// no formula for them; the formulas are SURVEY.md Appendix A (A1)-(A5), the readings
// are SURVEY.md 8(c) A1-A22, restated in DESIGN.md.  Pins: tests/test_oracle_pins.py.
//
// Parity status: every function below is pinned (P1-P13).
//
// Conventions:
//   * Rydberg atomic units, kappa = sqrt(z), Im kappa >= 0                       (A4, A5)
//   * complex Y_lm, Condon-Shortley phase, L = l(l+1)+m                          (A2)
//   * Gaunt C(L,L',L'') = Int Y_L^* Y_L' Y_L''^* dOmega                          (App. A)
//   * g0^{ij}_{LL'} = -4 pi i kappa sum_{l''} i^{l-l'+l''} h_{l''}(kappa R)
//                     Y_{l'',m'-m}(Rhat) C(L,L',(l'',m'-m)),  R = R_i - R_j     (A1, A3)
//   * t_l^{-1} = -kappa / (sin(delta_l) e^{i delta_l})                           (A2 of App. A)
//   * M column-major, ld = n, central site (API site 0) in the LAST block        (A13, A18)
//   * spin-canted within-site index s*kmax + L                                   (A11)
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

typedef std::complex<double> cd;
const double PI = 3.14159265358979323846264338327950288;

// ---------------------------------------------------------------- Legendre / harmonics

// Associated Legendre P_l^m(x), m >= 0, with Condon-Shortley phase (-1)^m, by the
// textbook upward recurrence in l starting from P_m^m.
double assoc_legendre(int l, int m, double x) {
    double pmm = 1.0;
    if (m > 0) {
        double s = std::sqrt((1.0 - x) * (1.0 + x));
        double f = 1.0;
        for (int i = 1; i <= m; ++i) { pmm *= -f * s; f += 2.0; }
    }
    if (l == m) return pmm;
    double pmmp1 = x * (2 * m + 1) * pmm;
    if (l == m + 1) return pmmp1;
    double pll = 0.0;
    for (int ll = m + 2; ll <= l; ++ll) {
        pll = (x * (2 * ll - 1) * pmmp1 - (ll + m - 1) * pmm) / (ll - m);
        pmm = pmmp1; pmmp1 = pll;
    }
    return pll;
}

double factorial(int n) { double f = 1.0; for (int i = 2; i <= n; ++i) f *= i; return f; }

// Y_lm(theta,phi) = sqrt((2l+1)/(4pi) (l-m)!/(l+m)!) P_l^m(cos theta) e^{i m phi};
// Y_{l,-m} = (-1)^m conj(Y_lm).                                       (reading A2)
cd ylm_angles(int l, int m, double costh, double phi) {
    int am = m < 0 ? -m : m;
    double norm = std::sqrt((2 * l + 1) / (4.0 * PI) * factorial(l - am) / factorial(l + am));
    cd y = norm * assoc_legendre(l, am, costh) * cd(std::cos(am * phi), std::sin(am * phi));
    if (m < 0) { y = std::conj(y); if (am & 1) y = -y; }
    return y;
}

// all Y_L(Rhat), L = l(l+1)+m, l <= lmax, from a (not necessarily unit) vector
void ylm_vec(int lmax, const double* v, cd* out) {
    double r = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    double costh = v[2] / r;
    double phi = std::atan2(v[1], v[0]);
    for (int l = 0; l <= lmax; ++l)
        for (int m = -l; m <= l; ++m) out[l * (l + 1) + m] = ylm_angles(l, m, costh, phi);
}

// Spherical Hankel functions of the first kind, h_0..h_lmax, upward recurrence
// (App. A: h_0 = -i e^{ix}/x, h_1 = -(1 + i/x) e^{ix}/x, h_{l+1} = (2l+1)/x h_l - h_{l-1}).
void hankel1(int lmax, cd x, cd* h) {
    const cd I(0.0, 1.0);
    cd e = std::exp(I * x);
    h[0] = -I * e / x;
    if (lmax >= 1) h[1] = -(1.0 + I / x) * e / x;
    for (int l = 1; l < lmax; ++l) h[l + 1] = double(2 * l + 1) / x * h[l] - h[l - 1];
}

// ---------------------------------------------------------------- Gaunt by quadrature

// Gauss-Legendre nodes/weights on (-1,1) by Newton iteration on P_n.
void gauss_legendre(int n, std::vector<double>& x, std::vector<double>& w) {
    x.resize(n); w.resize(n);
    for (int i = 0; i < n; ++i) {
        double z = std::cos(PI * (i + 0.75) / (n + 0.5));
        double pp = 0.0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 1; j <= n; ++j) { double p3 = p2; p2 = p1; p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j; }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            double dz = p1 / pp;
            z -= dz;
            if (std::fabs(dz) < 1e-16) break;
        }
        x[i] = z; w[i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

// C(L,L',L'') = Int Y_L^*(O) Y_L'(O) Y_L''^*(O) dO, Gauss-Legendre in cos(theta)
// (2 lmax_total + 2 nodes) x uniform phi (4 lmax_total + 2 nodes): exact to rounding for
// these band-limited integrands.
cd gaunt_quadrature(int l, int m, int lp, int mp, int lpp, int mpp) {
    int lt = l; if (lp > lt) lt = lp; if (lpp > lt) lt = lpp;
    int ng = 2 * lt + 2, nphi = 4 * lt + 2;
    std::vector<double> x, w; gauss_legendre(ng, x, w);
    cd acc = 0.0;
    for (int a = 0; a < ng; ++a)
        for (int b = 0; b < nphi; ++b) {
            double phi = 2.0 * PI * b / nphi;
            cd f = std::conj(ylm_angles(l, m, x[a], phi)) * ylm_angles(lp, mp, x[a], phi) *
                   std::conj(ylm_angles(lpp, mpp, x[a], phi));
            acc += w[a] * (2.0 * PI / nphi) * f;
        }
    return acc;
}

// Dense Gaunt table for the structure constants: G[(L*kmax + L')*nl2 + L''],
// L,L' < (lmax+1)^2, L'' < (2 lmax+1)^2.  Real parts stored (imaginary parts vanish; pin P13
// checks this through gaunt_quadrature directly).
struct GauntTable {
    int lmax, kmax, nl2;
    std::vector<double> g;
};

GauntTable build_gaunt(int lmax) {
    GauntTable t; t.lmax = lmax; t.kmax = (lmax + 1) * (lmax + 1); t.nl2 = (2 * lmax + 1) * (2 * lmax + 1);
    t.g.assign((size_t)t.kmax * t.kmax * t.nl2, 0.0);
    // tabulate Y on the quadrature grid once (same quadrature as gaunt_quadrature, max order)
    int lt = 2 * lmax, ng = 2 * lt + 2, nphi = 4 * lt + 2;
    std::vector<double> x, w; gauss_legendre(ng, x, w);
    std::vector<cd> Y((size_t)ng * nphi * t.nl2);
    for (int a = 0; a < ng; ++a)
        for (int b = 0; b < nphi; ++b)
            for (int l = 0; l <= lt; ++l)
                for (int m = -l; m <= l; ++m)
                    Y[((size_t)a * nphi + b) * t.nl2 + l * (l + 1) + m] = ylm_angles(l, m, x[a], 2.0 * PI * b / nphi);
    for (int L = 0; L < t.kmax; ++L)
        for (int Lp = 0; Lp < t.kmax; ++Lp)
            for (int Lpp = 0; Lpp < t.nl2; ++Lpp) {
                cd acc = 0.0;
                for (int a = 0; a < ng; ++a)
                    for (int b = 0; b < nphi; ++b) {
                        const cd* y = &Y[((size_t)a * nphi + b) * t.nl2];
                        acc += w[a] * (2.0 * PI / nphi) * std::conj(y[L]) * y[Lp] * std::conj(y[Lpp]);
                    }
                t.g[((size_t)L * t.kmax + Lp) * t.nl2 + Lpp] = acc.real();
            }
    return t;
}

const GauntTable& gaunt_cached(int lmax) {
    static std::vector<GauntTable*> cache;   // pointers: entries never move
    const GauntTable* hit = nullptr;
#pragma omp critical(gaunt_cache)
    {
        for (auto* t : cache) if (t->lmax == lmax) hit = t;
        if (!hit) { cache.push_back(new GauntTable(build_gaunt(lmax))); hit = cache.back(); }
    }
    return *hit;
}

void l_m_of(int L, int& l, int& m) { l = 0; while ((l + 1) * (l + 1) <= L) ++l; m = L - l * (l + 1); }

cd ipow(int p) { switch (((p % 4) + 4) % 4) { case 0: return cd(1, 0); case 1: return cd(0, 1); case 2: return cd(-1, 0); default: return cd(0, -1); } }

// ---------------------------------------------------------------- g0 block, eq. (A1)

// out[L + kmax*L'] = g0_{LL'}(R; kappa), R = R_i - R_j (row site minus column site).
void g0_block(int lmax, const double* R, cd kappa, cd* out) {
    const GauntTable& T = gaunt_cached(lmax);
    int kmax = T.kmax, nl2 = T.nl2;
    double r = std::sqrt(R[0] * R[0] + R[1] * R[1] + R[2] * R[2]);
    std::vector<cd> h(2 * lmax + 1), Y(nl2);
    hankel1(2 * lmax, kappa * r, h.data());
    ylm_vec(2 * lmax, R, Y.data());
    const cd pref = cd(0.0, -4.0 * PI) * kappa;   // -4 pi i kappa
    for (int L = 0; L < kmax; ++L) {
        int l, m; l_m_of(L, l, m);
        for (int Lp = 0; Lp < kmax; ++Lp) {
            int lp, mp; l_m_of(Lp, lp, mp);
            cd s = 0.0;
            for (int lpp = std::abs(l - lp); lpp <= l + lp; lpp += 2) {
                int mpp = mp - m;
                if (std::abs(mpp) > lpp) continue;
                int Lpp = lpp * (lpp + 1) + mpp;
                s += ipow(l - lp + lpp) * h[lpp] * Y[Lpp] * T.g[((size_t)L * kmax + Lp) * nl2 + Lpp];
            }
            out[L + (size_t)kmax * Lp] = pref * s;
        }
    }
}

// ---------------------------------------------------------------- single-site t^{-1}

// t_l = -(1/kappa) sin(delta_l) e^{i delta_l}  (BASELINE.json configs[0]);  t_l^{-1} = -kappa/(sin d e^{i d})
cd tinv_of(cd delta, cd kappa) { return -kappa / (std::sin(delta) * std::exp(cd(0, 1) * delta)); }

// ---------------------------------------------------------------- assembly of M, eq. (A4)

// M (column-major n x n) for one item.  site_pos[n_sites][3], species[n_sites],
// delta[2][n_spin][lmax+1], moment[n_sites][3] (used iff canted), z = energy.
void assemble_M(int n_sites, int lmax, int canted, const double* site_pos, const int32_t* species,
                const cd* delta, const double* moment, cd z, cd* M) {
    int kmax = (lmax + 1) * (lmax + 1), nspin = canted ? 2 : 1, k = kmax * nspin, n = n_sites * k;
    cd kappa = std::sqrt(z);                       // principal root; Im z >= 0 => Im kappa >= 0 (A4)
    if (kappa.imag() < 0) kappa = -kappa;
    for (size_t i = 0; i < (size_t)n * n; ++i) M[i] = 0.0;
    std::vector<cd> blk((size_t)kmax * kmax);
    auto blockpos = [&](int s) { return (s == 0 ? n_sites - 1 : s - 1) * k; };   // central last (A18)
    for (int si = 0; si < n_sites; ++si)
        for (int sj = 0; sj < n_sites; ++sj) {
            int r0 = blockpos(si), c0 = blockpos(sj);
            if (si == sj) {
                const cd* d = delta + (size_t)species[si] * nspin * (lmax + 1);
                for (int L = 0; L < kmax; ++L) {
                    int l, m; l_m_of(L, l, m);
                    if (!canted) {
                        M[(r0 + L) + (size_t)n * (c0 + L)] = tinv_of(d[l], kappa);
                    } else {
                        // (A3): t^{-1} = 1/2 (a+b) x 1 + 1/2 (a-b) x (sigma . e)
                        cd a = tinv_of(d[l], kappa), b = tinv_of(d[(lmax + 1) + l], kappa);
                        const double* e = moment + 3 * si;
                        cd hs = 0.5 * (a + b), hd = 0.5 * (a - b);
                        M[(r0 + L) + (size_t)n * (c0 + L)] = hs + hd * e[2];
                        M[(r0 + kmax + L) + (size_t)n * (c0 + kmax + L)] = hs - hd * e[2];
                        M[(r0 + L) + (size_t)n * (c0 + kmax + L)] = hd * cd(e[0], -e[1]);
                        M[(r0 + kmax + L) + (size_t)n * (c0 + L)] = hd * cd(e[0], e[1]);
                    }
                }
            } else {
                double R[3] = { site_pos[3 * si] - site_pos[3 * sj], site_pos[3 * si + 1] - site_pos[3 * sj + 1],
                                site_pos[3 * si + 2] - site_pos[3 * sj + 2] };
                g0_block(lmax, R, kappa, blk.data());
                for (int s = 0; s < nspin; ++s)
                    for (int Lp = 0; Lp < kmax; ++Lp)
                        for (int L = 0; L < kmax; ++L)
                            M[(r0 + s * kmax + L) + (size_t)n * (c0 + s * kmax + Lp)] = -blk[L + (size_t)kmax * Lp];
            }
        }
}

// ---------------------------------------------------------------- dense elimination

template <class R> struct cx { typedef std::complex<R> type; };

// Gaussian elimination with UNRESTRICTED partial pivoting on the augmented system [A | B]
// (A n x n, B n x nrhs, both column-major, both overwritten), then back-substitution;
// B returns X = A^{-1} B.  Returns 0 or the 1-based step at which a zero pivot was met.
// This is the textbook "LU then solve" route of PAPER.md:92.
template <class R>
int gauss_solve(int n, int nrhs, std::complex<R>* A, std::complex<R>* B) {
    typedef std::complex<R> C;
    for (int j = 0; j < n; ++j) {
        int p = j; R best = std::abs(A[j + (size_t)n * j]);
        for (int i = j + 1; i < n; ++i) { R v = std::abs(A[i + (size_t)n * j]); if (v > best) { best = v; p = i; } }
        if (!(best > R(0))) return j + 1;
        if (p != j) {
            for (int c = j; c < n; ++c) std::swap(A[j + (size_t)n * c], A[p + (size_t)n * c]);
            for (int c = 0; c < nrhs; ++c) std::swap(B[j + (size_t)n * c], B[p + (size_t)n * c]);
        }
        C piv = A[j + (size_t)n * j];
        for (int i = j + 1; i < n; ++i) A[i + (size_t)n * j] /= piv;
        for (int c = j + 1; c < n; ++c) {
            C u = A[j + (size_t)n * c];
            C* col = A + (size_t)n * c; const C* lcol = A + (size_t)n * j;
            for (int i = j + 1; i < n; ++i) col[i] -= lcol[i] * u;
        }
        for (int c = 0; c < nrhs; ++c) {
            C u = B[j + (size_t)n * c];
            C* col = B + (size_t)n * c; const C* lcol = A + (size_t)n * j;
            for (int i = j + 1; i < n; ++i) col[i] -= lcol[i] * u;
        }
    }
    for (int c = 0; c < nrhs; ++c) {
        C* x = B + (size_t)n * c;
        for (int i = n - 1; i >= 0; --i) {
            C s = x[i];
            for (int j2 = i + 1; j2 < n; ++j2) s -= A[i + (size_t)n * j2] * x[j2];
            x[i] = s / A[i + (size_t)n * i];
        }
    }
    return 0;
}

// tau00 by the textbook route: X = M^{-1} E (E = last k columns of I_n), tau00 = last k rows of X.
// If X_out != null the whole n x k block column is returned too.
template <class R>
int tau00_full(int n, int k, const cd* M, cd* tau, cd* X_out) {
    typedef std::complex<R> C;
    std::vector<C> A((size_t)n * n), B((size_t)n * k, C(0));
    for (size_t i = 0; i < (size_t)n * n; ++i) A[i] = C((R)M[i].real(), (R)M[i].imag());
    for (int c = 0; c < k; ++c) B[(n - k + c) + (size_t)n * c] = C(1);
    int info = gauss_solve<R>(n, k, A.data(), B.data());
    if (info) return info;
    for (int c = 0; c < k; ++c)
        for (int r = 0; r < k; ++r) {
            C v = B[(n - k + r) + (size_t)n * c];
            tau[r + (size_t)k * c] = cd((double)v.real(), (double)v.imag());
        }
    if (X_out)
        for (size_t i = 0; i < (size_t)n * k; ++i) X_out[i] = cd((double)B[i].real(), (double)B[i].imag());
    return 0;
}

// Second, independent route: eliminate the first n-k columns
// with pivots restricted to rows [j, n-k); the trailing k x k block is then the Schur complement
// D - C A^{-1} B, and tau00 is its inverse (computed with gauss_solve on [S | I]).
int tau00_schur(int n, int k, const cd* Min, cd* tau) {
    std::vector<cd> A(Min, Min + (size_t)n * n);
    int ne = n - k;
    for (int j = 0; j < ne; ++j) {
        int p = j; double best = std::abs(A[j + (size_t)n * j]);
        for (int i = j + 1; i < ne; ++i) { double v = std::abs(A[i + (size_t)n * j]); if (v > best) { best = v; p = i; } }
        if (!(best > 0.0)) return j + 1;
        if (p != j) for (int c = j; c < n; ++c) std::swap(A[j + (size_t)n * c], A[p + (size_t)n * c]);
        cd piv = A[j + (size_t)n * j];
        for (int i = j + 1; i < n; ++i) A[i + (size_t)n * j] /= piv;
        for (int c = j + 1; c < n; ++c) {
            cd u = A[j + (size_t)n * c];
            for (int i = j + 1; i < n; ++i) A[i + (size_t)n * c] -= A[i + (size_t)n * j] * u;
        }
    }
    std::vector<cd> S((size_t)k * k), E((size_t)k * k, cd(0));
    for (int c = 0; c < k; ++c) { for (int r = 0; r < k; ++r) S[r + (size_t)k * c] = A[(ne + r) + (size_t)n * (ne + c)]; E[c + (size_t)k * c] = 1.0; }
    int info = gauss_solve<double>(k, k, S.data(), E.data());
    if (info) return ne + info;
    std::memcpy(tau, E.data(), sizeof(cd) * k * k);
    return 0;
}

// Brute force: full inverse by Gauss-Jordan with partial pivoting (pin P6).
int inverse_gauss_jordan(int n, const cd* Min, cd* inv) {
    std::vector<cd> A(Min, Min + (size_t)n * n);
    for (size_t i = 0; i < (size_t)n * n; ++i) inv[i] = 0.0;
    for (int i = 0; i < n; ++i) inv[i + (size_t)n * i] = 1.0;
    for (int j = 0; j < n; ++j) {
        int p = j; double best = std::abs(A[j + (size_t)n * j]);
        for (int i = j + 1; i < n; ++i) { double v = std::abs(A[i + (size_t)n * j]); if (v > best) { best = v; p = i; } }
        if (!(best > 0.0)) return j + 1;
        if (p != j) for (int c = 0; c < n; ++c) { std::swap(A[j + (size_t)n * c], A[p + (size_t)n * c]); std::swap(inv[j + (size_t)n * c], inv[p + (size_t)n * c]); }
        cd piv = A[j + (size_t)n * j];
        for (int c = 0; c < n; ++c) { A[j + (size_t)n * c] /= piv; inv[j + (size_t)n * c] /= piv; }
        for (int i = 0; i < n; ++i) {
            if (i == j) continue;
            cd f = A[i + (size_t)n * j];
            if (f == cd(0)) continue;
            for (int c = 0; c < n; ++c) { A[i + (size_t)n * c] -= f * A[j + (size_t)n * c]; inv[i + (size_t)n * c] -= f * inv[j + (size_t)n * c]; }
        }
    }
    return 0;
}

// FP64 LU (kept) + iterative refinement with the residual accumulated in long double
// -- the parity variant for the large configs.
int tau00_refined(int n, int k, const cd* M, int n_refine, cd* tau, cd* X_out) {
    typedef std::complex<long double> CL;
    std::vector<cd> LU(M, M + (size_t)n * n);
    std::vector<int> piv(n);
    for (int j = 0; j < n; ++j) {
        int p = j; double best = std::abs(LU[j + (size_t)n * j]);
        for (int i = j + 1; i < n; ++i) { double v = std::abs(LU[i + (size_t)n * j]); if (v > best) { best = v; p = i; } }
        if (!(best > 0.0)) return j + 1;
        piv[j] = p;
        if (p != j) for (int c = 0; c < n; ++c) std::swap(LU[j + (size_t)n * c], LU[p + (size_t)n * c]);
        cd pv = LU[j + (size_t)n * j];
        for (int i = j + 1; i < n; ++i) LU[i + (size_t)n * j] /= pv;
        for (int c = j + 1; c < n; ++c) {
            cd u = LU[j + (size_t)n * c];
            cd* col = LU.data() + (size_t)n * c; const cd* lcol = LU.data() + (size_t)n * j;
            for (int i = j + 1; i < n; ++i) col[i] -= lcol[i] * u;
        }
    }
    auto lu_solve = [&](cd* b) {       // b <- M^{-1} b for one column
        for (int j = 0; j < n; ++j) { if (piv[j] != j) std::swap(b[j], b[piv[j]]); }
        for (int j = 0; j < n; ++j) { cd u = b[j]; for (int i = j + 1; i < n; ++i) b[i] -= LU[i + (size_t)n * j] * u; }
        for (int j = n - 1; j >= 0; --j) { b[j] /= LU[j + (size_t)n * j]; cd u = b[j]; for (int i = 0; i < j; ++i) b[i] -= LU[i + (size_t)n * j] * u; }
    };
    std::vector<cd> X((size_t)n * k, cd(0)), r(n);
    for (int c = 0; c < k; ++c) { X[(n - k + c) + (size_t)n * c] = 1.0; lu_solve(&X[(size_t)n * c]); }
    for (int it = 0; it < n_refine; ++it)
        for (int c = 0; c < k; ++c) {
            std::vector<CL> acc(n, CL(0));
            acc[n - k + c] = CL(1);
            for (int j = 0; j < n; ++j) {
                CL xj((long double)X[j + (size_t)n * c].real(), (long double)X[j + (size_t)n * c].imag());
                const cd* col = M + (size_t)n * j;
                for (int i = 0; i < n; ++i) acc[i] -= CL((long double)col[i].real(), (long double)col[i].imag()) * xj;
            }
            for (int i = 0; i < n; ++i) r[i] = cd((double)acc[i].real(), (double)acc[i].imag());
            lu_solve(r.data());
            for (int i = 0; i < n; ++i) X[i + (size_t)n * c] += r[i];
        }
    for (int c = 0; c < k; ++c) for (int rr = 0; rr < k; ++rr) tau[rr + (size_t)k * c] = X[(n - k + rr) + (size_t)n * c];
    if (X_out) std::memcpy(X_out, X.data(), sizeof(cd) * (size_t)n * k);
    return 0;
}

}  // namespace

// ================================================================== C entry points (ctypes)
extern "C" {

// complex values cross the boundary as interleaved (re,im) doubles.

void orc_gaunt_quadrature(int l, int m, int lp, int mp, int lpp, int mpp, double* out2) {
    cd c = gaunt_quadrature(l, m, lp, mp, lpp, mpp); out2[0] = c.real(); out2[1] = c.imag();
}
// dense table [kmax][kmax][(2lmax+1)^2] of real Gaunt numbers
void orc_gaunt_table(int lmax, double* out) { const GauntTable& t = gaunt_cached(lmax); std::memcpy(out, t.g.data(), sizeof(double) * t.g.size()); }
void orc_ylm(int lmax, const double* v3, double* out) { ylm_vec(lmax, v3, reinterpret_cast<cd*>(out)); }
void orc_hankel1(int lmax, const double* x2, double* out) { hankel1(lmax, cd(x2[0], x2[1]), reinterpret_cast<cd*>(out)); }
void orc_g0_block(int lmax, const double* R3, const double* kappa2, double* out) { g0_block(lmax, R3, cd(kappa2[0], kappa2[1]), reinterpret_cast<cd*>(out)); }
void orc_tinv(const double* delta2, const double* kappa2, double* out2) {
    cd t = tinv_of(cd(delta2[0], delta2[1]), cd(kappa2[0], kappa2[1])); out2[0] = t.real(); out2[1] = t.imag();
}
void orc_assemble_M(int n_sites, int lmax, int canted, const double* site_pos, const int32_t* species,
                    const double* delta, const double* moment, const double* z2, double* M) {
    assemble_M(n_sites, lmax, canted, site_pos, species, reinterpret_cast<const cd*>(delta), moment, cd(z2[0], z2[1]),
               reinterpret_cast<cd*>(M));
}
// precision: 0 = double, 1 = long double
int orc_tau00_full(int n, int k, const double* M, int precision, double* tau, double* X_out) {
    if (precision == 1) return tau00_full<long double>(n, k, reinterpret_cast<const cd*>(M), reinterpret_cast<cd*>(tau), reinterpret_cast<cd*>(X_out));
    return tau00_full<double>(n, k, reinterpret_cast<const cd*>(M), reinterpret_cast<cd*>(tau), reinterpret_cast<cd*>(X_out));
}
int orc_tau00_schur(int n, int k, const double* M, double* tau) { return tau00_schur(n, k, reinterpret_cast<const cd*>(M), reinterpret_cast<cd*>(tau)); }
int orc_tau00_refined(int n, int k, const double* M, int n_refine, double* tau, double* X_out) {
    return tau00_refined(n, k, reinterpret_cast<const cd*>(M), n_refine, reinterpret_cast<cd*>(tau), reinterpret_cast<cd*>(X_out));
}
int orc_inverse_gauss_jordan(int n, const double* M, double* inv) { return inverse_gauss_jordan(n, reinterpret_cast<const cd*>(M), reinterpret_cast<cd*>(inv)); }

// Whole path for a batch, as the timed CPU baseline runs it: assemble M, then the FP64 textbook
// solve.  OpenMP over batch items, one item per thread.  Returns the
// number of items with non-zero info.  mode: 0 = tau00_full<double>, 1 = <long double>, 2 = schur.
int orc_tau00_batched(int batch, int n_sites, int lmax, int canted, const double* site_pos, const int32_t* species,
                      const double* delta, const double* moment, const double* z, int mode, double* tau_out, int* info) {
    int kmax = (lmax + 1) * (lmax + 1), k = kmax * (canted ? 2 : 1), n = n_sites * k;
    gaunt_cached(lmax);
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : bad)
    for (int b = 0; b < batch; ++b) {
        std::vector<cd> M((size_t)n * n);
        assemble_M(n_sites, lmax, canted, site_pos + (size_t)b * n_sites * 3, species + (size_t)b * n_sites,
                   reinterpret_cast<const cd*>(delta), moment + (size_t)b * n_sites * 3, cd(z[2 * b], z[2 * b + 1]), M.data());
        cd* tau = reinterpret_cast<cd*>(tau_out) + (size_t)b * k * k;
        int inf;
        if (mode == 1) inf = tau00_full<long double>(n, k, M.data(), tau, nullptr);
        else if (mode == 2) inf = tau00_schur(n, k, M.data(), tau);
        else inf = tau00_full<double>(n, k, M.data(), tau, nullptr);
        info[b] = inf; if (inf) ++bad;
    }
    return bad;
}

int orc_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// the tau part of the contour integral of eq. (2)/(3): for every central atom a,
//   out_a = sum_q w_q tau00_{a,q},   q over the n_e contour points, w_q = quadrature weight * dz/dq (complex).
// tau [n_atoms][n_e][kk], w [n_e], out [n_atoms][kk]; plain loops in the order of the definition.
void orc_contour_sum(int n_atoms, int n_e, int kk, const double* tau, const double* w, double* out) {
    const cd* T = reinterpret_cast<const cd*>(tau); const cd* W = reinterpret_cast<const cd*>(w); cd* O = reinterpret_cast<cd*>(out);
    for (int a = 0; a < n_atoms; ++a)
        for (int e = 0; e < kk; ++e) {
            cd s(0.0, 0.0);
            for (int q = 0; q < n_e; ++q) s += W[q] * T[((size_t)a * n_e + q) * kk + e];
            O[(size_t)a * kk + e] = s;
        }
}

}  // extern "C"
