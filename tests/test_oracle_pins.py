"""Pins for the CPU oracle.

Each test checks oracle/ against something OTHER than itself: closed forms, the
addition theorem evaluated with scipy's Bessel functions and harmonics, library
(LAPACK via numpy) inverses, algebraic identities, symmetries, the paper's
printed ranks.  No CUDA here.
"""
import math
import os

import numpy as np
import pytest
import scipy.special as sps

import oracle
import synth_liz as sl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def lm(L):
    l = int(math.isqrt(L))
    return l, L - l * (l + 1)


def scipy_ylm(l, m, v):
    v = np.asarray(v, float)
    r = np.linalg.norm(v)
    theta = math.acos(v[2] / r)
    phi = math.atan2(v[1], v[0])
    return complex(sps.sph_harm_y(l, m, theta, phi))


def relF(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


# ----------------------------------------------------------------- building blocks

def test_ylm_matches_scipy_and_is_orthonormal():
    rng = np.random.default_rng(1)
    for _ in range(5):
        v = rng.standard_normal(3)
        y = oracle.ylm(8, v)
        ref = np.array([scipy_ylm(*lm(L), v) for L in range(81)])
        assert np.max(np.abs(y - ref)) < 5e-14
    # poles: only m = 0 survives
    y = oracle.ylm(4, [0, 0, 2.0])
    for L in range(25):
        l, m = lm(L)
        exp = math.sqrt((2 * l + 1) / (4 * math.pi)) if m == 0 else 0.0
        assert abs(y[L] - exp) < 1e-15
    y = oracle.ylm(4, [0, 0, -1.0])
    for L in range(25):
        l, m = lm(L)
        exp = (-1) ** l * math.sqrt((2 * l + 1) / (4 * math.pi)) if m == 0 else 0.0
        assert abs(y[L] - exp) < 1e-15


def test_hankel_matches_scipy_complex_argument():
    for x in [3.6 + 0.0j, 4.2 + 0.3j, 0.5 + 3.0j, 11.0 + 0.01j, 2.0 + 2.0j]:
        h = oracle.hankel1(16, x)
        n = np.arange(17)
        ref = sps.spherical_jn(n, x) + 1j * sps.spherical_yn(n, x)
        assert np.max(np.abs(h - ref) / np.abs(ref)) < 1e-10
    # closed forms h0, h1
    x = 1.7 + 0.4j
    h = oracle.hankel1(1, x)
    assert abs(h[0] - (-1j) * np.exp(1j * x) / x) < 1e-16
    assert abs(h[1] - (-(1 + 1j / x) * np.exp(1j * x) / x)) < 1e-16


def test_P13_gaunt_closed_forms_selection_rules_and_counts():
    ns = {"sqrt": math.sqrt, "pi": math.pi}
    with open(os.path.join(GOLD, "gaunt_closed_forms.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if not line:
                continue
            p = line.split()
            q = [int(t) for t in p[:6]]
            exp = eval(" ".join(p[6:]), ns)
            got = oracle.gaunt_quadrature(*q)
            assert abs(got - exp) < 2e-15, (q, got, exp)
    # 498 / 1463 (L,L',l'') triples pass the selection rules; 6 / 10 of them vanish
    # accidentally (e.g. the 3j symbol (2 3 3; 0 2 -2) = 0), leaving 492 / 1453 non-zero numbers.
    for lmax, count, count_nz in ((3, 498, 492), (4, 1463, 1453)):
        T = oracle.gaunt_table(lmax)
        kmax = (lmax + 1) ** 2
        nz = 0
        n_allowed = 0
        for L in range(kmax):
            l, m = lm(L)
            for Lp in range(kmax):
                lp, mp = lm(Lp)
                row = T[L, Lp]
                for Lpp in range((2 * lmax + 1) ** 2):
                    lpp, mpp = lm(Lpp)
                    allowed = (mpp == mp - m and (l + lp + lpp) % 2 == 0 and abs(l - lp) <= lpp <= l + lp)
                    if not allowed:
                        assert abs(row[Lpp]) < 1e-14
                n_allowed += sum(1 for lpp in range(abs(l - lp), l + lp + 1, 2) if abs(mp - m) <= lpp)
                nz += sum(1 for lpp in range(abs(l - lp), l + lp + 1, 2)
                          if abs(mp - m) <= lpp and abs(row[lpp * (lpp + 1) + mp - m]) > 1e-12)
        assert n_allowed == count and nz == count_nz


def test_gaunt_vs_scipy_numeric_integration():
    # independent route: scipy harmonics on a fine product grid
    x, w = np.polynomial.legendre.leggauss(24)
    phi = 2 * np.pi * np.arange(48) / 48
    th = np.arccos(x)
    TH, PH = np.meshgrid(th, phi, indexing="ij")
    W = w[:, None] * (2 * np.pi / 48)
    rng = np.random.default_rng(5)
    T = oracle.gaunt_table(3)
    for _ in range(40):
        L, Lp = rng.integers(0, 16, 2)
        l, m = lm(L)
        lp, mp = lm(Lp)
        lpp = rng.integers(abs(l - lp), l + lp + 1)
        mpp = mp - m
        if abs(mpp) > lpp:
            continue
        val = np.sum(W * np.conj(sps.sph_harm_y(l, m, TH, PH)) * sps.sph_harm_y(lp, mp, TH, PH)
                     * np.conj(sps.sph_harm_y(lpp, mpp, TH, PH)))
        assert abs(val.imag) < 1e-14
        assert abs(T[L, Lp, lpp * (lpp + 1) + mpp] - val.real) < 1e-14
        assert abs(oracle.gaunt_quadrature(l, m, lp, mp, lpp, mpp) - val) < 1e-14


# ----------------------------------------------------------------- g0: P1, P2, P7, P8

KAPPAS = [0.8367 + 0j, np.sqrt(-0.3 + 0.02j), np.sqrt(0.1 + 0.6j)]


def test_P1_g0_s_channel_closed_form():
    R = np.array([1.3, -2.2, 4.1])
    r = np.linalg.norm(R)
    for kap in KAPPAS:
        g = oracle.g0_block(3, R, kap)
        assert abs(g[0, 0] - (-np.exp(1j * kap * r) / r)) < 1e-15


def test_P2_two_centre_expansion_of_free_green_function():
    """G0(rho - rho' + R) = sum_{LL'} j_l(k rho) Y_L(rho^) g0_LL'(R) j_l'(k rho') Y_L'^*(rho'^),
    G0(x) = -exp(i k |x|)/(4 pi |x|).  Fixes every sign, phase and
    index convention of g0 at once; converges geometrically in the cut-off."""
    rng = np.random.default_rng(7)
    R = sl.site_positions(13)[3] - sl.site_positions(13)[0]      # a nearest-neighbour vector
    for kap in KAPPAS:
        errs = []
        rho = 0.35 * rng.standard_normal(3)
        rhop = 0.35 * rng.standard_normal(3)
        x = rho - rhop + R
        exact = -np.exp(1j * kap * np.linalg.norm(x)) / (4 * np.pi * np.linalg.norm(x))
        for lt in (2, 4, 6):
            g = oracle.g0_block(lt, R, kap)
            k = (lt + 1) ** 2
            a = np.array([sps.spherical_jn(lm(L)[0], kap * np.linalg.norm(rho)) * scipy_ylm(*lm(L), rho) for L in range(k)])
            b = np.array([sps.spherical_jn(lm(L)[0], kap * np.linalg.norm(rhop)) * np.conj(scipy_ylm(*lm(L), rhop)) for L in range(k)])
            errs.append(abs(a @ g @ b - exact) / abs(exact))
        assert errs[0] < 3e-2 and errs[1] < 3e-4 and errs[2] < 1e-5, errs      # SURVEY probe B1: 4e-3, 1e-5, 4e-7
        assert errs[2] < errs[1] < errs[0]


def test_P7_P8_parity_and_reciprocity():
    R = np.array([2.1, 0.7, -3.3])
    for kap in KAPPAS:
        g = oracle.g0_block(4, R, kap)
        gm = oracle.g0_block(4, -R, kap)
        tol = 1e-14 * np.abs(g).max()
        for L in range(25):
            l, m = lm(L)
            for Lp in range(25):
                lp, mp = lm(Lp)
                assert abs(gm[L, Lp] - (-1) ** (l + lp) * g[L, Lp]) < tol          # P7
                Lb, Lpb = l * (l + 1) - m, lp * (lp + 1) - mp
                assert abs(g[L, Lp] - (-1) ** (m + mp) * gm[Lpb, Lb]) < tol        # P8


# ----------------------------------------------------------------- t^{-1} and assembly

def test_tinv_closed_form():
    for d, kap in [(0.7 + 0.02j, 0.8 + 0.1j), (1.4 + 0.05j, 0.3 + 0.7j)]:
        got = oracle.tinv(d, kap)
        assert abs(got - (-kap / np.tan(d) + 1j * kap)) < 1e-14       # -k cot d + i k
        t = -(1 / kap) * np.sin(d) * np.exp(1j * d)                   # configs[0]
        assert abs(got * t - 1) < 1e-14


def _item(cfg, b=0, batch=None):
    batch = batch or sl.make_batch(cfg)
    return batch, dict(n_sites=cfg.n_sites, lmax=cfg.lmax, canted=cfg.spin_canted, site_pos=batch.site_pos[b],
                       species=batch.species[b], delta=batch.delta, moment=batch.moment_dir[b], z=batch.z[b])


def test_assembly_structure_and_central_last():
    cfg = sl.CONFIGS["T"]
    batch, it = _item(cfg, 5)
    M = oracle.assemble_M(**it)
    k, n = cfg.k, cfg.n
    assert M.shape == (n, n)
    kap = np.sqrt(batch.z[5])
    for s in range(cfg.n_sites):
        blk = (cfg.n_sites - 1 if s == 0 else s - 1) * k
        D = M[blk:blk + k, blk:blk + k]
        exp = np.diag([oracle.tinv(batch.delta[batch.species[5, s], 0, lm(L)[0]], kap) for L in range(k)])
        assert np.array_equal(D, exp)                       # g0^{ii} = 0
    # off-diagonal block (site 3 row, site 0 col) = -g0(R_3 - R_0), stored at rows of 3, cols of LAST block
    g = oracle.g0_block(3, batch.site_pos[5, 3] - batch.site_pos[5, 0], kap)
    assert np.allclose(M[2 * k:3 * k, n - k:], -g, rtol=0, atol=1e-15)


def test_P12_shapes_from_paper_and_configs():
    with open(os.path.join(GOLD, "paper_shapes.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if not line:
                continue
            nl, lmax, c, rank = (int(t) for t in line.split())
            assert nl * (lmax + 1) ** 2 * (2 if c else 1) == rank
            assert nl in sl.FCC_SHELL_CLOSURES
    for key, n in zip("TMPCH", (208, 880, 2160, 4320, 6750)):
        assert sl.CONFIGS[key].n == n
    pts = sl.fcc_liz_lattice_points(135)
    assert tuple(pts[0]) == (0, 0, 0) and len({tuple(p) for p in pts}) == 135
    d2 = (pts ** 2).sum(1)
    assert np.all(np.diff(d2) >= 0) and d2[12] == 2 and d2[13] == 4 and d2[134] == 14
    # nearest-neighbour distance a/sqrt(2) = 5.0777 Bohr (A5)
    assert abs(np.linalg.norm(sl.site_positions(13)[1]) - 5.077705) < 1e-5


# ----------------------------------------------------------------- solves: P3-P6, P9

def test_P3_single_site_limit():
    cfg = sl.custom_config(1, 3, False)
    batch, it = _item(cfg)
    M = oracle.assemble_M(**it)
    kap = np.sqrt(batch.z[0])
    t = np.array([-(1 / kap) * np.sin(batch.delta[batch.species[0, 0], 0, lm(L)[0]])
                  * np.exp(1j * batch.delta[batch.species[0, 0], 0, lm(L)[0]]) for L in range(16)])
    for f in (oracle.tau00_full, oracle.tau00_schur):
        tau = f(M, 16)
        assert relF(tau, np.diag(t)) < 1e-15
    # canted single site: tau = rotated 2k x 2k t
    cfg = sl.custom_config(1, 2, True)
    batch, it = _item(cfg)
    M = oracle.assemble_M(**it)
    tau = oracle.tau00_full(M, 18)
    kap = np.sqrt(batch.z[0])
    sp = batch.species[0, 0]
    e = batch.moment_dir[0, 0]
    ta = np.array([-(1 / kap) * np.sin(batch.delta[sp, 0, lm(L)[0]]) * np.exp(1j * batch.delta[sp, 0, lm(L)[0]]) for L in range(9)])
    tb = np.array([-(1 / kap) * np.sin(batch.delta[sp, 1, lm(L)[0]]) * np.exp(1j * batch.delta[sp, 1, lm(L)[0]]) for L in range(9)])
    sig = np.array([[e[2], e[0] - 1j * e[1]], [e[0] + 1j * e[1], -e[2]]])
    exp = np.kron(np.eye(2), np.diag((ta + tb) / 2)) + np.kron(sig, np.diag((ta - tb) / 2))
    assert relF(tau, exp) < 1e-14


@pytest.mark.parametrize("q", [0, 16, 31])
def test_P4_P5_P6_P9_tiny_liz(q):
    cfg = sl.CONFIGS["T"]
    batch, it = _item(cfg, q)
    M = oracle.assemble_M(**it)
    n, k = cfg.n, cfg.k
    tau, X = oracle.tau00_full(M, k, want_X=True)
    inv_np = np.linalg.inv(M)                                  # LAPACK: independent library routine
    assert relF(tau, inv_np[n - k:, n - k:]) < 1e-12           # definition: central block of M^{-1}
    assert relF(oracle.inverse_gauss_jordan(M), inv_np) < 1e-12            # P6
    assert relF(oracle.tau00_schur(M, k), tau) < 1e-12                     # P4
    assert relF(oracle.tau00_full(M, k, "long double"), tau) < 1e-12
    assert relF(oracle.tau00_refined(M, k, 2), oracle.tau00_full(M, k, "long double")) < 1e-14
    E = np.zeros((n, k)); E[n - k:] = np.eye(k)
    assert np.linalg.norm(M @ X - E) / (np.linalg.norm(M) * np.linalg.norm(X)) < 1e-15   # P5
    # P9: [(I - t g0)^{-1} t]_00 with t, g0 rebuilt here from the oracle's blocks
    tinv_d = np.diag(M).copy()
    g0 = np.diag(tinv_d) - M
    t = np.diag(1 / tinv_d)
    alt = np.linalg.solve(np.eye(n) - t @ g0, t)[n - k:, n - k:]
    assert relF(tau, alt) < 1e-12


def test_brute_force_random_matrices_all_routes():
    A = sl.random_dense_matrices(3, 57, seed=11)
    for b in range(3):
        M = A[b].T                                             # [row, col]
        ref = np.linalg.inv(M)[-9:, -9:]
        assert relF(oracle.tau00_full(M, 9), ref) < 1e-12
        assert relF(oracle.tau00_schur(M, 9), ref) < 1e-12
        assert relF(oracle.tau00_refined(M, 9, 1), ref) < 1e-12
    # a matrix that NEEDS pivoting (zero leading entry)
    M = np.array([[0, 2, 1], [1, 1, 0], [3, 0, 1]], dtype=complex)
    assert relF(oracle.tau00_full(M, 1), np.linalg.inv(M)[-1:, -1:]) < 1e-15
    assert relF(oracle.tau00_schur(M, 1), np.linalg.inv(M)[-1:, -1:]) < 1e-15


def test_singular_matrix_reports_info():
    M = np.ones((4, 4), dtype=complex)
    with pytest.raises(np.linalg.LinAlgError):
        oracle.tau00_full(M, 1)


# ----------------------------------------------------------------- spin canting: P10, P11

def test_P10_collinear_moments_decouple():
    cfg = sl.custom_config(13, 2, True, n_energies=2)
    batch, it = _item(cfg, 1)
    it["moment"] = np.tile([0.0, 0.0, 1.0], (13, 1))
    tau = oracle.tau00_full(oracle.assemble_M(**it), 18)
    assert np.all(tau[:9, 9:] == 0) and np.all(tau[9:, :9] == 0)
    for s in range(2):
        it1 = dict(it, canted=False, delta=batch.delta[:, s:s + 1, :])
        t1 = oracle.tau00_full(oracle.assemble_M(**it1), 9)
        assert relF(tau[9 * s:9 * s + 9, 9 * s:9 * s + 9], t1) < 1e-13


def test_P11_global_spin_rotation_covariance():
    cfg = sl.custom_config(13, 2, True, n_energies=2)
    batch, it = _item(cfg, 0)
    tau = oracle.tau00_full(oracle.assemble_M(**it), 18)
    # SU(2) element for a rotation by angle a about axis u;  U (sigma.e) U^+ = sigma.(Rot e)
    a, u = 0.83, np.array([0.3, -0.5, 0.81]); u /= np.linalg.norm(u)
    sx = np.array([[0, 1], [1, 0]], complex); sy = np.array([[0, -1j], [1j, 0]]); sz = np.array([[1, 0], [0, -1]], complex)
    U = math.cos(a / 2) * np.eye(2) - 1j * math.sin(a / 2) * (u[0] * sx + u[1] * sy + u[2] * sz)
    Kx = np.array([[0, -u[2], u[1]], [u[2], 0, -u[0]], [-u[1], u[0], 0]])
    Rot = np.eye(3) + math.sin(a) * Kx + (1 - math.cos(a)) * Kx @ Kx
    it2 = dict(it, moment=batch.moment_dir[0] @ Rot.T)
    tau2 = oracle.tau00_full(oracle.assemble_M(**it2), 18)
    UU = np.kron(U, np.eye(9))
    assert relF(tau2, UU @ tau @ UU.conj().T) < 1e-13


# ----------------------------------------------------------------- batched driver + generator

def test_batched_driver_matches_single_item_calls():
    cfg = sl.custom_config(13, 2, True, n_atoms=2, n_energies=3)
    batch = sl.make_batch(cfg)
    tau, info = oracle.tau00_batched(batch, "double")
    assert not info.any() and tau.shape == (6, 18, 18)
    for b in (0, 4):
        _, it = _item(cfg, b, batch)
        assert relF(tau[b], oracle.tau00_full(oracle.assemble_M(**it), 18)) < 1e-15
    tau_s, _ = oracle.tau00_batched(batch, "schur")
    assert relF(tau_s, tau) < 1e-12


def test_generator_recipe():
    r = sl.SplitMix64(0)
    assert r.next_u64() == 0xE220A8397B1DCDAF                   # published SplitMix64 test vector, seed 0
    z = sl.contour_energies("semicircle", 32)
    assert abs(z[0].real + 0.5) < 2e-3 and abs(z[-1].real - 0.7) < 2e-3 and np.all(z.imag > 0)
    assert abs(z.imag.min() - 2.58e-3) < 1e-4 and abs(np.abs(z).min() - 0.5) < 5e-3      # A6
    za = sl.contour_energies("arc", 24)
    assert abs(za[0] - (0.5251 + 0.4235j)) < 1e-3 and abs(za[-1] - (0.7 + 0.0011j)) < 1e-3   # A7
    b = sl.make_batch("T")
    assert b.z.shape == (32,) and b.species.shape == (32, 13) and set(np.unique(b.species)) <= {0, 1}
    d = sl.phase_shift_table(sl.CONFIGS["H"])
    assert np.all(d[1, :, 2].real == 1.4) and d.shape == (2, 2, 5)
    assert np.all((d.real > 0) & (d.real < 1.5) & (d.imag > 0) & (d.imag < 0.05))
    bc = sl.make_batch("C", n_atoms=1, n_energies=2)
    assert np.allclose(np.linalg.norm(bc.moment_dir, axis=-1), 1.0)


# ------------------------------------------------------------------ contour reduction

def test_contour_sum_closed_forms():
    """sum_q w_q tau(z_q) against integrals known in closed form (eq. (2): an energy integral up to E_F
    taken along the contour): polynomials int_{-0.5}^{0.7} z^m dz = (0.7^{m+1} - (-0.5)^{m+1})/(m+1), and a simple
    pole, where the arc over the pole differs from the straight path by -2 pi i (clockwise closed contour), while a
    pole outside the half disc gives the principal-branch logarithm.  Fixes weights, node order and the reduction."""
    for kind, npts, z_end in (("semicircle", 32, -0.5 + 0j), ("arc", 24, 0.1 + 0.6 * np.exp(1j * np.pi / 4))):
        z = sl.contour_energies(kind, npts)
        w = sl.contour_weights(kind, npts)
        # a 3 x 2 "matrix" of monomials per atom, two atoms with different prefactors
        tau = np.zeros((2, npts, 3, 2), dtype=np.complex128)
        for a in range(2):
            for i in range(3):
                for j in range(2):
                    tau[a, :, i, j] = (a + 1.5) * z ** (2 * i + j)
        out = oracle.contour_sum(tau, w)
        for a in range(2):
            for i in range(3):
                for j in range(2):
                    m = 2 * i + j
                    exact = (a + 1.5) * (0.7 ** (m + 1) - z_end ** (m + 1)) / (m + 1)
                    assert abs(out[a, i, j] - exact) < 2e-14
    z = sl.contour_energies("semicircle", 32)
    w = sl.contour_weights("semicircle", 32)
    for z0, winding in ((0.1 + 0.3j, -2j * np.pi), (0.1 + 0.9j, 0.0), (0.2 - 0.4j, 0.0)):
        val = oracle.contour_sum((1.0 / (z - z0))[None, :, None], w)[0, 0]
        exact = np.log(0.7 - z0) - np.log(-0.5 - z0) + winding
        assert abs(val - exact) < 2e-6          # truncation error of the 32-point rule for a pole 0.3 away (seen: 4e-7)
    # linearity and the order of the energy axis: a weight vector with a single 1 picks that energy's tau
    rng = np.random.default_rng(5)
    tau = rng.standard_normal((3, 7, 4, 4)) + 1j * rng.standard_normal((3, 7, 4, 4))
    for q in (0, 3, 6):
        e = np.zeros(7, dtype=np.complex128); e[q] = 1.0
        assert np.array_equal(oracle.contour_sum(tau, e), tau[:, q])


def test_stored_full_size_values_are_well_formed():
    """tests/golden/tau00_full_size_*.txt (written by make_golden_full_size.py from oracle/ alone): header matches the
    workload's shape, every (row, col) present once, finite; and the route that wrote them (FP64 LU + long-double
    refinement) agrees with the long-double textbook route on a case small enough to run here."""
    import glob
    files = sorted(glob.glob(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "tau00_full_size_*.txt")))
    assert files, "run tests/golden/make_golden_full_size.py"
    for path in files:
        with open(path) as f:
            head = f.readline().split()
            cfg = sl.CONFIGS[head[1]]
            assert int(head[3]) == cfg.n and int(head[4]) == cfg.k and 0 <= int(head[2]) < cfg.batch
            seen = set()
            for line in f:
                r, c, re, im = line.split()
                seen.add((int(r), int(c)))
                assert np.isfinite(float(re)) and np.isfinite(float(im))
            assert len(seen) == cfg.k * cfg.k
    cfg = sl.custom_config(19, 2, True, n_energies=2)
    b = sl.make_batch(cfg)
    M = oracle.assemble_M(cfg.n_sites, cfg.lmax, cfg.spin_canted, b.site_pos[1], b.species[1], b.delta, b.moment_dir[1], b.z[1])
    assert relF(oracle.tau00_refined(M, cfg.k, 3), oracle.tau00_full(M, cfg.k, "long double")) < 1e-14

