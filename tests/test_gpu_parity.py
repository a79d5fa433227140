"""GPU parity: the CUDA path (through the C ABI binding) against the CPU oracle, element by element
on the same seeded inputs.  Bars (BASELINE.json north_star):
relative Frobenius error <= 1e-10 on tau00, normwise residual <= 1e-12, assembled M within
1e-13 of the oracle's M relative to the largest entry of its site block."""
import os

import numpy as np
import pytest

import oracle
import synth_liz as sl

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TAU_TOL = 1e-10
RES_TOL = 1e-12
ASM_TOL = 1e-13


@pytest.fixture(scope="module")
def lt():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2308_16317_b200 as m
    m.lib()
    return m


def relF(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def gpu_M(lt, batch):
    cfg = batch.cfg
    delta, species, z, pos, mom = lt.device_inputs(batch)
    tinv, kappa = lt.lsms_tinv_from_phase_shifts(delta, species, z, cfg.lmax, cfg.n_sites, cfg.spin_canted, 2, batch.batch)
    M = lt.lsms_build_M_batched(tinv, pos, mom if cfg.spin_canted else None, kappa, cfg.lmax, cfg.n_sites,
                                cfg.spin_canted, batch.batch)
    return M, tinv, kappa


def oracle_M(batch, b):
    cfg = batch.cfg
    return oracle.assemble_M(cfg.n_sites, cfg.lmax, cfg.spin_canted, batch.site_pos[b], batch.species[b], batch.delta,
                             batch.moment_dir[b], batch.z[b])


def block_rel_err(Mg, Mo, k):
    """max over site blocks of max|diff| / max|oracle block| (blocks that are exactly zero must match exactly)"""
    n = Mo.shape[0]
    nb = n // k
    d = np.abs(Mg - Mo).reshape(nb, k, nb, k).max(axis=(1, 3))
    s = np.abs(Mo).reshape(nb, k, nb, k).max(axis=(1, 3))
    assert np.all(d[s == 0] == 0)
    return float((d[s > 0] / s[s > 0]).max())


def residual(M, X, k):
    """||M X - E||_F / (||M||_F ||X||_F), E = last k columns of I (reading A15)."""
    n = M.shape[0]
    E = np.zeros((n, k)); E[n - k:] = np.eye(k)
    return np.linalg.norm(M @ X - E) / (np.linalg.norm(M) * np.linalg.norm(X))


# ------------------------------------------------------------------ K1: t^{-1} and assembly

def test_tinv_and_kappa_parity(lt):
    batch = sl.make_batch("C", n_atoms=1, n_energies=32)
    _, tinv, kappa = gpu_M(lt, batch.select([0]))     # shapes only
    delta, species, z, pos, mom = lt.device_inputs(batch)
    tinv, kappa = lt.lsms_tinv_from_phase_shifts(delta, species, z, 3, 135, True, 2, 32)
    tinv, kappa = tinv.cpu().numpy(), kappa.cpu().numpy()
    assert np.max(np.abs(kappa - np.sqrt(batch.z))) < 1e-15 and np.all(kappa.imag >= 0)
    for b in (0, 17, 31):
        for s in (0, 5, 134):
            for sp in range(2):
                for l in range(4):
                    ref = oracle.tinv(batch.delta[batch.species[b, s], sp, l], np.sqrt(batch.z[b]))
                    assert abs(tinv[b, s, sp, l] - ref) <= 4e-15 * abs(ref)


@pytest.mark.parametrize("key,items", [("T", list(range(32))), ("M", [0, 31, 200, 511])])
def test_assembly_parity_noncanted(lt, key, items):
    batch = sl.make_batch(key).select(items)
    M, _, _ = gpu_M(lt, batch)
    Mg = M.cpu().numpy().transpose(0, 2, 1)
    for i in range(len(items)):
        assert block_rel_err(Mg[i], oracle_M(batch, i), batch.cfg.k) < ASM_TOL


def test_assembly_parity_canted_and_high_l(lt):
    for key, items in (("C", [0, 63]), ("H", [0, 23])):
        batch = sl.make_batch(key).select(items)
        M, _, _ = gpu_M(lt, batch)
        for i in range(len(items)):
            Mg = M[i].cpu().numpy().T
            assert block_rel_err(Mg, oracle_M(batch, i), batch.cfg.k) < ASM_TOL
        del M
        torch.cuda.empty_cache()


def test_assembly_small_lmax_range(lt):
    for lmax, canted in ((0, False), (1, True), (2, False), (5, False)):
        cfg = sl.custom_config(13, lmax, canted, n_energies=3)
        batch = sl.make_batch(cfg)
        M, _, _ = gpu_M(lt, batch)
        Mg = M.cpu().numpy().transpose(0, 2, 1)
        for i in range(3):
            assert block_rel_err(Mg[i], oracle_M(batch, i), cfg.k) < ASM_TOL


def test_shared_g0_assembly_is_identical_to_per_item_assembly(lt):
    """one g0 evaluation per energy shared by all central atoms of a lattice.  Same arithmetic per
    element, so the matrices must be bit-identical to the per-item assembly (which is itself checked against the
    oracle above); plain and spin-canted (per-item moments and t^-1 on the site diagonal), and one oracle block check."""
    for cfg in (sl.custom_config(19, 3, False, n_atoms=3, n_energies=5), sl.custom_config(13, 2, True, n_atoms=4, n_energies=3),
                sl.custom_config(13, 4, False, n_atoms=2, n_energies=2)):
        batch = sl.make_batch(cfg)
        delta, species, z, pos, mom = lt.device_inputs(batch)
        tinv, kappa = lt.lsms_tinv_from_phase_shifts(delta, species, z, cfg.lmax, cfg.n_sites, cfg.spin_canted, 2, batch.batch)
        momd = mom if cfg.spin_canted else None
        M_item = lt.lsms_build_M_batched(tinv, pos, momd, kappa, cfg.lmax, cfg.n_sites, cfg.spin_canted, batch.batch)
        M_shared = lt.lsms_build_M_shared_g0_batched(tinv, pos, momd, kappa, cfg.lmax, cfg.n_sites, cfg.spin_canted,
                                                     cfg.n_atoms, cfg.n_energies)
        torch.cuda.synchronize()
        assert torch.equal(torch.view_as_real(M_item), torch.view_as_real(M_shared))
        b = batch.batch - 1                                         # last atom, last energy
        assert block_rel_err(M_shared[b].cpu().numpy().T, oracle_M(batch, b), cfg.k) < ASM_TOL


# ------------------------------------------------------------------ whole path, element-wise

def test_tau00_tiny_full_batch(lt):
    batch = sl.make_batch("T")
    tau, info, _ = lt.tau00_from_liz_batch(batch)
    assert not info.any()
    ref, oinfo = oracle.tau00_batched(batch, "long double")
    assert not oinfo.any()
    for b in range(32):
        assert relF(tau[b], ref[b]) < TAU_TOL
    assert max(relF(tau[b], ref[b]) for b in range(32)) < 1e-12     # expected ~1e-14 at cond ~1e3


def test_tau00_mid_sampled(lt):
    items = [0, 24, 31, 100, 255, 256, 480, 511]
    batch = sl.make_batch("M").select(items)
    tau, info, _ = lt.tau00_from_liz_batch(batch)
    assert not info.any()
    ref, _ = oracle.tau00_batched(batch, "long double")
    for b in range(len(items)):
        assert relF(tau[b], ref[b]) < TAU_TOL


def test_tau00_reduced_high_l_canted(lt):
    """H-like (lmax=4, canted, near-resonant Au d channel) at 19 sites: n = 950, k = 50 -- ragged in
    every blocking (n-k = 900 = 14*64 + 4; inner panels of 16 and 4)."""
    cfg = sl.LizConfig("high-l", 4, 19, 4, True, 1, 6, "arc")
    batch = sl.make_batch(cfg)
    tau, info, _ = lt.tau00_from_liz_batch(batch)
    assert not info.any()
    ref, _ = oracle.tau00_batched(batch, "long double")
    for b in range(batch.batch):
        assert relF(tau[b], ref[b]) < TAU_TOL


def test_tau00_full_size_mid_batch_residual_every_item(lt):
    """Full M batch (512 items) in the launch configuration bench.py times: info == 0 everywhere, and the
    residual of the verification export on every item (computed with torch on the device: test-side
    cuBLAS, not the product path)."""
    batch = sl.make_batch("M")
    cfg = batch.cfg
    M, _, _ = gpu_M(lt, batch)
    X, info = lt.lsms_solve_central_column_batched(M, cfg.n_sites, cfg.kmax, False, batch.batch)
    tau, info2 = lt.lsms_tau00_batched(M.clone(), cfg.n_sites, cfg.kmax, False, batch.batch)
    torch.cuda.synchronize()
    assert not info.cpu().numpy().any() and not info2.cpu().numpy().any()
    n, k = cfg.n, cfg.k
    Mm = M.transpose(1, 2)                     # [b, row, col]
    Xm = X.transpose(1, 2)                     # [b, n, k]
    R = torch.bmm(Mm, Xm)
    R[:, n - k:, :] -= torch.eye(k, dtype=R.dtype, device=R.device)
    res = torch.linalg.matrix_norm(R) / (torch.linalg.matrix_norm(Mm) * torch.linalg.matrix_norm(Xm))
    assert float(res.max()) < RES_TOL
    # tau00 is the central block of X
    assert float((Xm[:, n - k:, :] - tau.transpose(1, 2)).abs().max()) == 0.0


@pytest.mark.parametrize("key,items,mode", [("P", [0, 24, 31, 56, 64, 88, 120, 127], "double"),
                                             ("C", [0, 16, 24, 31, 32, 47, 56, 63], "double")])
def test_tau00_production_sizes_sampled(lt, key, items, mode):
    """2160^2 and 4320^2 (the north-star sizes): eight sampled items each (first and last energy of every atom, the
    worst-conditioned contour point q = 24) against the oracle's textbook route, which runs one item per host
    thread, plus the residual of the central block column for the same items on the host."""
    batch = sl.make_batch(key).select(items)
    cfg = batch.cfg
    M, _, _ = gpu_M(lt, batch)
    X, info = lt.lsms_solve_central_column_batched(M, cfg.n_sites, cfg.kmax, cfg.spin_canted, batch.batch)
    Mh = [M[i].cpu().numpy().T for i in range(len(items))]
    Xh = [X[i].cpu().numpy().T for i in range(len(items))]
    tau, info2 = lt.lsms_tau00_batched(M, cfg.n_sites, cfg.kmax, cfg.spin_canted, batch.batch)
    torch.cuda.synchronize()
    tau = tau.cpu().numpy().transpose(0, 2, 1)
    assert not info.cpu().numpy().any() and not info2.cpu().numpy().any()
    for i in range(len(items)):
        assert residual(Mh[i], Xh[i], cfg.k) < RES_TOL
    ref, oinfo = oracle.tau00_batched(batch, mode)
    assert not oinfo.any()
    for i in range(len(items)):
        assert relF(tau[i], ref[i]) < TAU_TOL, (key, items[i], relF(tau[i], ref[i]))


def test_tau00_high_l_full_size_properties(lt):
    """6750^2 (the paper's CoCrFeMnNi rank): the oracle needs ~10 min per item, so parity is
    by properties that hold at any size: M equals the oracle's M (cheap), the residual of the central block
    column is <= 1e-12, and tau00 equals the central block of that column."""
    items = [0, 23]
    batch = sl.make_batch("H").select(items)
    cfg = batch.cfg
    M, _, _ = gpu_M(lt, batch)
    X, info = lt.lsms_solve_central_column_batched(M, cfg.n_sites, cfg.kmax, True, batch.batch)
    torch.cuda.synchronize()
    assert not info.cpu().numpy().any()
    for i in range(len(items)):
        Mo = oracle_M(batch, i)
        assert block_rel_err(M[i].cpu().numpy().T, Mo, cfg.k) < ASM_TOL
        assert residual(Mo, X[i].cpu().numpy().T, cfg.k) < RES_TOL


@pytest.mark.parametrize("key,item", [("H", 0), ("H", 23), ("N", 23), ("C", 24)])
def test_tau00_full_size_against_stored_oracle_values(lt, key, item):
    """Element-wise parity at full size where the oracle needs minutes per item: tau00 of single items of the
    largest workloads (H item 0 is the worst-conditioned matrix of all configs, cond_1 ~ 1.6e6) against values the
    oracle wrote into tests/golden/ (tests/golden/make_golden_full_size.py: oracle.assemble_M + FP64 LU with
    long-double iterative refinement; nothing there comes from the CUDA path)."""
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", f"tau00_full_size_{key}_{item}.txt")
    with open(path) as f:
        head = f.readline().split()
        assert head[1] == key and int(head[2]) == item
        n, k = int(head[3]), int(head[4])
        ref = np.zeros((k, k), dtype=np.complex128)
        for line in f:
            r, c, re, im = line.split()
            ref[int(r), int(c)] = complex(float(re), float(im))
    batch = sl.make_batch(key).select([item])
    assert batch.cfg.n == n and batch.cfg.k == k
    tau, info, _ = lt.tau00_from_liz_batch(batch)
    assert not info.any()
    assert relF(tau[0], ref) < TAU_TOL, relF(tau[0], ref)


@pytest.mark.parametrize("key,item", [("N", 23), ("NC", 0)])
def test_tau00_paper_niau_shapes_properties(lt, key, item):
    """the paper's own NiAu ranks 6225 and 12450 (N_LIZ = 249, l_max = 4).  Same
    property checks as the high-l case: assembled M equals the oracle's M block by block, the central block column
    solves M X = E to <= 1e-12, and tau00 is the central block of X (checked against lsms_tau00_batched itself)."""
    batch = sl.make_batch(key).select([item])
    cfg = batch.cfg
    assert cfg.n == {"N": 6225, "NC": 12450}[key]
    M, _, _ = gpu_M(lt, batch)
    X, info = lt.lsms_solve_central_column_batched(M, cfg.n_sites, cfg.kmax, cfg.spin_canted, 1)
    torch.cuda.synchronize()
    assert not info.cpu().numpy().any()
    Mo = oracle_M(batch, 0)
    assert block_rel_err(M[0].cpu().numpy().T, Mo, cfg.k) < ASM_TOL
    Xh = X[0].cpu().numpy().T
    assert residual(Mo, Xh, cfg.k) < RES_TOL
    tau, info2 = lt.lsms_tau00_batched(M, cfg.n_sites, cfg.kmax, cfg.spin_canted, 1)      # overwrites M
    torch.cuda.synchronize()
    assert not info2.cpu().numpy().any()
    assert relF(tau[0].cpu().numpy().T, Xh[cfg.n - cfg.k:, :]) < 1e-12


# ------------------------------------------------------------------ direct input to lsms_tau00_batched

@pytest.mark.parametrize("n_sites,kmax,canted", [(7, 9, False), (37, 1, False), (1, 16, False), (2, 4, True),
                                                  (33, 4, False), (5, 25, True), (129, 1, False)])
def test_random_matrices_vs_lapack(lt, n_sites, kmax, canted):
    k = kmax * (2 if canted else 1)
    n = n_sites * k
    A = sl.random_dense_matrices(5, n, seed=100 + n)
    M = torch.from_numpy(A).cuda()
    tau, info = lt.lsms_tau00_batched(M, n_sites, kmax, canted, 5)
    torch.cuda.synchronize()
    tau = tau.cpu().numpy().transpose(0, 2, 1)
    assert not info.cpu().numpy().any()
    for b in range(5):
        ref = np.linalg.inv(A[b].T)[n - k:, n - k:]
        assert relF(tau[b], ref) < 1e-11


def test_needs_pivoting_and_singular_info(lt):
    # zero on the leading diagonal: fails without row interchanges
    n_sites, kmax = 6, 4
    n = 24
    rng = np.random.default_rng(3)
    A = rng.standard_normal((3, n, n)) + 1j * rng.standard_normal((3, n, n))
    for j in range(n):
        A[0, j, j] = 0.0                       # column-major storage: [b, col, row]
    A[2, 5, :] = 0.0                           # column 5 identically zero -> exact zero pivot at step 6
    M = torch.from_numpy(np.ascontiguousarray(A)).cuda()
    tau, info = lt.lsms_tau00_batched(M, n_sites, kmax, False, 3)
    torch.cuda.synchronize()
    info = info.cpu().numpy()
    tau = tau.cpu().numpy().transpose(0, 2, 1)
    assert info[0] == 0 and info[1] == 0
    for b in (0, 1):
        assert relF(tau[b], np.linalg.inv(A[b].T)[n - 4:, n - 4:]) < 1e-11
    assert info[2] == 6


def test_blocking_parameters_do_not_change_the_result(lt):
    batch = sl.make_batch("T").select([0, 9])
    ref, _ = oracle.tau00_batched(batch, "long double")
    try:
        for nb, ib in ((16, 4), (32, 16), (48, 12), (96, 16), (64, 7)):
            lt.lsms_set_blocking(nb, ib)
            tau, info, _ = lt.tau00_from_liz_batch(batch)
            assert not info.any()
            assert max(relF(tau[b], ref[b]) for b in range(2)) < 1e-12
    finally:
        lt.lsms_set_blocking(0, 0)


def test_lookahead_on_and_off_give_identical_results(lt):
    """The look-ahead split of the Schur update only re-orders independent tiles: bitwise equal tau00."""
    batch = sl.make_batch("M").select([3, 300])
    try:
        lt.lsms_set_lookahead(False)
        tau0, info0, _ = lt.tau00_from_liz_batch(batch)
        lt.lsms_set_lookahead(True)
        tau1, info1, _ = lt.tau00_from_liz_batch(batch)
    finally:
        lt.lsms_set_lookahead(True)
    assert not info0.any() and not info1.any()
    assert np.array_equal(tau0, tau1)


@pytest.mark.parametrize("variant", [-1, 0, 1])
def test_panel_kernel_variants_match_oracle(lt, variant):
    """Every K2 variant (L2-resident columns, register-blocked sub-panels with 256 / 512 threads) against the
    oracle on a tiny LIZ, a ragged random matrix (w and sub-panel tails) and a mid LIZ (several row chunks)."""
    try:
        lt.lsms_set_panel_variant(variant)
        batch = sl.make_batch("T").select([0, 17, 31])
        ref, _ = oracle.tau00_batched(batch, "long double")
        tau, info, _ = lt.tau00_from_liz_batch(batch)
        assert not info.any()
        assert max(relF(tau[b], ref[b]) for b in range(3)) < 1e-12
        for n_sites, kmax in ((23, 9), (41, 4), (150, 9)):
            n = n_sites * kmax
            A = sl.random_dense_matrices(2, n, seed=700 + n)             # column-major storage: [b, col, row]
            tau, info = lt.lsms_tau00_batched(torch.from_numpy(A).cuda(), n_sites, kmax, False, 2)
            torch.cuda.synchronize()
            assert not info.cpu().numpy().any()
            tau = tau.cpu().numpy().transpose(0, 2, 1)
            for b in range(2):
                assert relF(tau[b], np.linalg.inv(A[b].T)[n - kmax:, n - kmax:]) < 1e-10
        mid = sl.make_batch("M").select([5, 400])
        refm, _ = oracle.tau00_batched(mid, "long double")
        taum, infom, _ = lt.tau00_from_liz_batch(mid)
        assert not infom.any()
        assert max(relF(taum[b], refm[b]) for b in range(2)) < 1e-10
    finally:
        lt.lsms_set_panel_variant(1)


@pytest.mark.parametrize("cl", [2, 4, 8])
def test_panel_cluster_kernel_matches_one_cta_kernel_and_oracle(lt, cl):
    """K2 with a cluster of cl CTAs per matrix: same pivots and arithmetic as the one-CTA kernel, so tau00 must be
    bit-identical to it; also against the oracle / LAPACK on a tiny LIZ, ragged random matrices (rows not a multiple
    of the cluster's thread count, sub-panel tails) and a singular matrix (info)."""
    try:
        batch = sl.make_batch("T").select([0, 31])
        ref, _ = oracle.tau00_batched(batch, "long double")
        lt.lsms_set_panel_cluster(1)
        tau1, info1, _ = lt.tau00_from_liz_batch(batch)
        lt.lsms_set_panel_cluster(cl)
        tau, info, _ = lt.tau00_from_liz_batch(batch)
        assert not info.any() and not info1.any()
        assert np.array_equal(tau, tau1)
        assert max(relF(tau[b], ref[b]) for b in range(2)) < 1e-12
        for n_sites, kmax in ((23, 9), (150, 9), (131, 16)):
            n = n_sites * kmax
            A = sl.random_dense_matrices(2, n, seed=900 + n)             # column-major storage: [b, col, row]
            lt.lsms_set_panel_cluster(1)
            t1, i1 = lt.lsms_tau00_batched(torch.from_numpy(A).cuda(), n_sites, kmax, False, 2)
            lt.lsms_set_panel_cluster(cl)
            t2, i2 = lt.lsms_tau00_batched(torch.from_numpy(A).cuda(), n_sites, kmax, False, 2)
            torch.cuda.synchronize()
            assert not i1.cpu().numpy().any() and not i2.cpu().numpy().any()
            assert torch.equal(torch.view_as_real(t1), torch.view_as_real(t2))
            t2 = t2.cpu().numpy().transpose(0, 2, 1)
            for b in range(2):
                assert relF(t2[b], np.linalg.inv(A[b].T)[n - kmax:, n - kmax:]) < 1e-10
        A = sl.random_dense_matrices(1, 24, seed=3)
        A[0, 5, :] = 0.0                           # column 5 identically zero -> exact zero pivot at step 6
        _, i3 = lt.lsms_tau00_batched(torch.from_numpy(A).cuda(), 6, 4, False, 1)
        torch.cuda.synchronize()
        assert int(i3.cpu().numpy()[0]) == 6
    finally:
        lt.lsms_set_panel_cluster(0)


def test_batch_groups_give_identical_results(lt):
    """Batch groups run the same per-item elimination on separate streams: bitwise equal tau00 for every
    group count, including counts that do not divide the batch and exceed it."""
    batch = sl.make_batch("T").select(list(range(11)))
    ref, _ = oracle.tau00_batched(batch, "long double")
    out = []
    try:
        for g in (1, 2, 3, 8):
            lt.lsms_set_groups(g)
            tau, info, _ = lt.tau00_from_liz_batch(batch)
            assert not info.any()
            out.append(tau)
        lt.lsms_set_groups(8)
        small = sl.make_batch("T").select([0, 5, 9])
        tau_s, info_s, _ = lt.tau00_from_liz_batch(small)
        assert not info_s.any()
    finally:
        lt.lsms_set_groups(0)
    for tau in out[1:]:
        assert np.array_equal(out[0], tau)
    assert max(relF(out[0][b], ref[b]) for b in range(11)) < 1e-10
    assert np.array_equal(tau_s, out[0][[0, 5, 9]])


def test_schur_update_alone_matches_numpy(lt):
    """K4 in isolation: C -= A B on ragged shapes (several tiles + tails in M, N and K; K of 1..6 chunks, so both the
    one-stage and the three-stage ring are exercised)."""
    if True:
        for n, c0, kk, nb in ((333, 10, 64, 2), (200, 0, 37, 2), (130, 3, 16, 2), (97, 40, 5, 2), (700, 20, 96, 3), (450, 7, 48, 5),
                              (1100, 0, 64, 1)):
            A = sl.random_dense_matrices(nb, n, seed=n)
            M = torch.from_numpy(A).cuda()
            lt.lsms_schur_update_batched(M, n, c0, kk, nb)
            torch.cuda.synchronize()
            out = M.cpu().numpy().transpose(0, 2, 1)
            for b in range(nb):
                ref = A[b].T.copy()
                r0 = c0 + kk
                ref[r0:, r0:] -= ref[r0:, c0:r0] @ ref[c0:r0, r0:]
                assert np.max(np.abs(out[b] - ref)) < 1e-12 * np.abs(ref).max() * kk


# ------------------------------------------------------------------ contour reduction

def test_contour_sum_matches_oracle(lt):
    """sum_q w_q tau00_{a,q} on the device vs the oracle's loop: the real tau00 of two tiny-LIZ atoms on the full
    32-point contour, plus ragged shapes (k*k not a multiple of the block, one energy, many atoms)."""
    cfg = sl.custom_config(13, 3, False, n_atoms=2, n_energies=32, index=0)
    batch = sl.make_batch(cfg)
    tau, info, _ = lt.tau00_from_liz_batch(batch)
    assert not info.any()
    w = sl.contour_weights("semicircle", 32)
    ref = oracle.contour_sum(tau.reshape(2, 32, cfg.k, cfg.k), w)
    tau_d = torch.from_numpy(np.ascontiguousarray(tau)).cuda()
    out = lt.lsms_contour_sum_batched(tau_d, torch.from_numpy(w).cuda(), 2, 32, cfg.k)
    torch.cuda.synchronize()
    assert relF(out.cpu().numpy(), ref) < 1e-14
    rng = np.random.default_rng(11)
    for na, ne, k in ((1, 1, 1), (5, 24, 50), (300, 3, 7), (2, 33, 13)):
        t = rng.standard_normal((na, ne, k, k)) + 1j * rng.standard_normal((na, ne, k, k))
        ww = rng.standard_normal(ne) + 1j * rng.standard_normal(ne)
        out = lt.lsms_contour_sum_batched(torch.from_numpy(t).cuda(), torch.from_numpy(ww).cuda(), na, ne, k)
        torch.cuda.synchronize()
        ref = oracle.contour_sum(t, ww)
        assert np.max(np.abs(out.cpu().numpy() - ref)) < 1e-13 * np.sqrt(ne) * np.abs(t).max() * np.abs(ww).max()


# ------------------------------------------------------------------ end-to-end host entry point

def test_host_entry_point_matches_device_path(lt):
    batch = sl.make_batch("T")
    cfg = batch.cfg
    hc = lt.HostCall(cfg.n_sites, cfg.lmax, cfg.spin_canted, 2, batch.batch)
    hc.load(batch)
    tau_h, info_h = hc.run()
    tau_d, info_d, _ = lt.tau00_from_liz_batch(batch)
    assert not info_h.numpy().any()
    assert np.array_equal(tau_h.numpy().transpose(0, 2, 1), tau_d)
    assert hc.h2d_bytes == batch.delta.nbytes + batch.species.nbytes + batch.z.nbytes + batch.site_pos.nbytes
    assert hc.d2h_bytes == 32 * 16 * 16 * 16 + 32 * 4
    assert lt.lsms_last_launch_count() > 10
