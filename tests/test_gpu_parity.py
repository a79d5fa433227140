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


@pytest.fixture()
def h(lt):
    """A fresh handle with default options for every test (the library has no process-wide state)."""
    hd = lt.lsms_create()
    yield hd
    torch.cuda.synchronize()
    hd.destroy()


def relF(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def max_abs_rel(a, b):
    """largest element-wise deviation relative to the largest reference element"""
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


def check_tau(tau, ref, tol=TAU_TOL, what=""):
    """north_star bar (relative Frobenius error) AND an element-wise bar, so that an error confined to a few
    elements cannot hide in the norm: max|diff| <= tol * max|ref|."""
    assert relF(tau, ref) < tol, (what, "rel. Frobenius", relF(tau, ref))
    assert max_abs_rel(tau, ref) < tol, (what, "max abs / max", max_abs_rel(tau, ref))


def gpu_M(lt, h, batch):
    cfg = batch.cfg
    delta, species, z, pos, mom = lt.device_inputs(batch)
    tinv, kappa, info0 = lt.lsms_tinv_from_phase_shifts(h, delta, species, z, cfg.lmax, cfg.n_sites, cfg.spin_canted, 2, batch.batch)
    M, info1 = lt.lsms_build_M_batched(h, tinv, pos, mom if cfg.spin_canted else None, kappa, cfg.lmax, cfg.n_sites,
                                       cfg.spin_canted, batch.batch)
    assert not info0.cpu().numpy().any() and not info1.cpu().numpy().any()
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

def test_tinv_and_kappa_parity(lt, h):
    batch = sl.make_batch("C", n_atoms=1, n_energies=32)
    _, tinv, kappa = gpu_M(lt, h, batch.select([0]))     # shapes only
    delta, species, z, pos, mom = lt.device_inputs(batch)
    tinv, kappa, _ = lt.lsms_tinv_from_phase_shifts(h, delta, species, z, 3, 135, True, 2, 32)
    tinv, kappa = tinv.cpu().numpy(), kappa.cpu().numpy()
    assert np.max(np.abs(kappa - np.sqrt(batch.z))) < 1e-15 and np.all(kappa.imag >= 0)
    for b in (0, 17, 31):
        for s in (0, 5, 134):
            for sp in range(2):
                for l in range(4):
                    ref = oracle.tinv(batch.delta[batch.species[b, s], sp, l], np.sqrt(batch.z[b]))
                    assert abs(tinv[b, s, sp, l] - ref) <= 4e-15 * abs(ref)


@pytest.mark.parametrize("key,items", [("T", list(range(32))), ("M", [0, 31, 200, 511])])
def test_assembly_parity_noncanted(lt, h, key, items):
    batch = sl.make_batch(key).select(items)
    M, _, _ = gpu_M(lt, h, batch)
    Mg = M.cpu().numpy().transpose(0, 2, 1)
    for i in range(len(items)):
        assert block_rel_err(Mg[i], oracle_M(batch, i), batch.cfg.k) < ASM_TOL


def test_assembly_parity_canted_and_high_l(lt, h):
    for key, items in (("C", [0, 63]), ("H", [0, 23])):
        batch = sl.make_batch(key).select(items)
        M, _, _ = gpu_M(lt, h, batch)
        for i in range(len(items)):
            Mg = M[i].cpu().numpy().T
            assert block_rel_err(Mg, oracle_M(batch, i), batch.cfg.k) < ASM_TOL
        del M
        torch.cuda.empty_cache()


def test_assembly_small_lmax_range(lt, h):
    for lmax, canted in ((0, False), (1, True), (2, False), (5, False)):
        cfg = sl.custom_config(13, lmax, canted, n_energies=3)
        batch = sl.make_batch(cfg)
        M, _, _ = gpu_M(lt, h, batch)
        Mg = M.cpu().numpy().transpose(0, 2, 1)
        for i in range(3):
            assert block_rel_err(Mg[i], oracle_M(batch, i), cfg.k) < ASM_TOL


def test_shared_g0_assembly_is_identical_to_per_item_assembly(lt, h):
    """one g0 evaluation per energy shared by all central atoms of a lattice.  Same arithmetic per
    element, so the matrices must be bit-identical to the per-item assembly (which is itself checked against the
    oracle above); plain and spin-canted (per-item moments and t^-1 on the site diagonal), and one oracle block check."""
    for cfg in (sl.custom_config(19, 3, False, n_atoms=3, n_energies=5), sl.custom_config(13, 2, True, n_atoms=4, n_energies=3),
                sl.custom_config(13, 4, False, n_atoms=2, n_energies=2)):
        batch = sl.make_batch(cfg)
        delta, species, z, pos, mom = lt.device_inputs(batch)
        tinv, kappa, _ = lt.lsms_tinv_from_phase_shifts(h, delta, species, z, cfg.lmax, cfg.n_sites, cfg.spin_canted, 2, batch.batch)
        momd = mom if cfg.spin_canted else None
        M_item, _ = lt.lsms_build_M_batched(h, tinv, pos, momd, kappa, cfg.lmax, cfg.n_sites, cfg.spin_canted, batch.batch)
        M_shared, _ = lt.lsms_build_M_shared_g0_batched(h, tinv, pos, momd, kappa, cfg.lmax, cfg.n_sites, cfg.spin_canted,
                                                     cfg.n_atoms, cfg.n_energies)
        torch.cuda.synchronize()
        assert torch.equal(torch.view_as_real(M_item), torch.view_as_real(M_shared))
        b = batch.batch - 1                                         # last atom, last energy
        assert block_rel_err(M_shared[b].cpu().numpy().T, oracle_M(batch, b), cfg.k) < ASM_TOL


# ------------------------------------------------------------------ whole path, element-wise

def test_tau00_tiny_full_batch(lt, h):
    batch = sl.make_batch("T")
    tau, info, _ = lt.tau00_from_liz_batch(h, batch)
    assert not info.any()
    ref, oinfo = oracle.tau00_batched(batch, "long double")
    assert not oinfo.any()
    for b in range(32):
        check_tau(tau[b], ref[b], 1e-12, ("T", b))              # expected ~1e-14 at cond ~1e3


def test_tau00_mid_sampled(lt, h):
    items = [0, 24, 31, 100, 255, 256, 480, 511]
    batch = sl.make_batch("M").select(items)
    tau, info, _ = lt.tau00_from_liz_batch(h, batch)
    assert not info.any()
    ref, _ = oracle.tau00_batched(batch, "long double")
    for b in range(len(items)):
        check_tau(tau[b], ref[b], TAU_TOL, ("M", items[b]))


def test_tau00_reduced_high_l_canted(lt, h):
    """H-like (lmax=4, canted, near-resonant Au d channel) at 19 sites: n = 950, k = 50 -- ragged in
    every blocking (n-k = 900 = 14*64 + 4; inner panels of 16 and 4); both schedules of the batch scheduler."""
    cfg = sl.LizConfig("high-l", 4, 19, 4, True, 1, 6, "arc")
    batch = sl.make_batch(cfg)
    ref, _ = oracle.tau00_batched(batch, "long double")
    for small in (1, 2):
        h.set("small_mode", small)
        tau, info, _ = lt.tau00_from_liz_batch(h, batch)
        assert not info.any()
        assert (lt.lsms_last_schedule(h) > 0) == (small == 2)
        for b in range(batch.batch):
            check_tau(tau[b], ref[b], TAU_TOL, ("high-l 19 sites", small, b))


def device_residuals(M, X, n, k):
    """||M X - E||_F / (||M||_F ||X||_F) of every item, on the device with torch (test-side cuBLAS, not the product path);
    M [b, col, row], X [b, col(k), row(n)] as the library stores them."""
    Mm, Xm = M.transpose(1, 2), X.transpose(1, 2)
    res = []
    for b0 in range(0, M.shape[0], 16):                     # chunks bound the temporaries
        R = torch.bmm(Mm[b0:b0 + 16], Xm[b0:b0 + 16])
        R[:, n - k:, :] -= torch.eye(k, dtype=R.dtype, device=R.device)
        res.append(torch.linalg.matrix_norm(R) / (torch.linalg.matrix_norm(Mm[b0:b0 + 16]) * torch.linalg.matrix_norm(Xm[b0:b0 + 16])))
    return torch.cat(res)


def test_tau00_full_size_mid_batch_residual_every_item(lt, h):
    """Full M batch (512 items) in the launch configuration bench.py times (default handle: lock-step, two batch groups,
    look-ahead): info == 0 everywhere, the residual of the verification export on every item, tau00 equal to the
    central block of X, and the one-launch small-matrix mode (one CTA per matrix, four matrices per SM) agreeing with
    the lock-step schedule on every item."""
    batch = sl.make_batch("M")
    cfg = batch.cfg
    n, k = cfg.n, cfg.k
    M, _, _ = gpu_M(lt, h, batch)
    X, info = lt.lsms_solve_central_column_batched(h, M, cfg.n_sites, cfg.kmax, False, batch.batch)
    tau, info2 = lt.lsms_tau00_batched(h, M.clone(), cfg.n_sites, cfg.kmax, False, batch.batch)
    sched = lt.lsms_last_schedule(h)
    h.set("small_mode", 2)
    tau_ls, info3 = lt.lsms_tau00_batched(h, M.clone(), cfg.n_sites, cfg.kmax, False, batch.batch)
    torch.cuda.synchronize()
    assert sched == 0 and lt.lsms_last_schedule(h) == 1
    assert not info.cpu().numpy().any() and not info2.cpu().numpy().any() and not info3.cpu().numpy().any()
    assert float(device_residuals(M, X, n, k).max()) < RES_TOL
    assert float((X[:, :, n - k:] - tau).abs().max()) == 0.0            # tau00 is the central block of X
    d = torch.linalg.matrix_norm(tau - tau_ls) / torch.linalg.matrix_norm(tau_ls)
    assert float(d.max()) < 1e-11                                      # two schedules, same pivots, different summation order


@pytest.mark.parametrize("key,items", [("P", [0, 24, 31, 56, 64, 88, 120, 127]), ("C", [0, 16, 24, 31, 32, 47, 56, 63])])
def test_tau00_production_full_batch(lt, h, key, items):
    """2160^2 and 4320^2 (the north-star sizes) as bench.py times them: the FULL batch (128 / 64 items) through a
    default handle -- two batch groups on separate streams with look-ahead --, info == 0 and the residual of the
    central block column on EVERY item (SURVEY 8(d) protocol, pin P5), and eight items (first and last energy of
    every atom, the worst-conditioned contour point q = 24) element by element against the oracle's textbook route."""
    batch = sl.make_batch(key)
    cfg = batch.cfg
    n, k, B = cfg.n, cfg.k, batch.batch
    M, _, _ = gpu_M(lt, h, batch)
    X, info = lt.lsms_solve_central_column_batched(h, M, cfg.n_sites, cfg.kmax, cfg.spin_canted, B)
    torch.cuda.synchronize()
    assert not info.cpu().numpy().any()
    res = device_residuals(M, X, n, k)
    assert float(res.max()) < RES_TOL, float(res.max())
    tau, info2 = lt.lsms_tau00_batched(h, M, cfg.n_sites, cfg.kmax, cfg.spin_canted, B)       # overwrites M
    torch.cuda.synchronize()
    assert lt.lsms_last_schedule(h) == 0 and h.get("groups") == 0 and h.get("lookahead") == 1
    assert not info2.cpu().numpy().any()
    assert float((X[:, :, n - k:] - tau).abs().max()) == 0.0
    tau = tau.cpu().numpy().transpose(0, 2, 1)
    del M, X
    torch.cuda.empty_cache()
    ref, oinfo = oracle.tau00_batched(batch.select(items), "double")
    assert not oinfo.any()
    for i, b in enumerate(items):
        check_tau(tau[b], ref[i], TAU_TOL, (key, b))


def test_tau00_high_l_full_size_properties(lt, h):
    """6750^2 (the paper's CoCrFeMnNi rank): the oracle needs ~10 min per item, so parity is
    by properties that hold at any size: M equals the oracle's M (cheap), the residual of the central block
    column is <= 1e-12, and tau00 equals the central block of that column."""
    items = [0, 23]
    batch = sl.make_batch("H").select(items)
    cfg = batch.cfg
    M, _, _ = gpu_M(lt, h, batch)
    X, info = lt.lsms_solve_central_column_batched(h, M, cfg.n_sites, cfg.kmax, True, batch.batch)
    torch.cuda.synchronize()
    assert not info.cpu().numpy().any()
    for i in range(len(items)):
        Mo = oracle_M(batch, i)
        assert block_rel_err(M[i].cpu().numpy().T, Mo, cfg.k) < ASM_TOL
        assert residual(Mo, X[i].cpu().numpy().T, cfg.k) < RES_TOL


def read_golden(key, item):
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", f"tau00_full_size_{key}_{item}.txt")
    with open(path) as f:
        head = f.readline().split()
        assert head[1] == key and int(head[2]) == item
        n, k = int(head[3]), int(head[4])
        ref = np.zeros((k, k), dtype=np.complex128)
        for line in f:
            r, c, re, im = line.split()
            ref[int(r), int(c)] = complex(float(re), float(im))
    return n, k, ref


@pytest.mark.parametrize("panel_cluster", [0, 1])
@pytest.mark.parametrize("key,item", [("H", 0), ("H", 23), ("N", 23), ("C", 24), ("P", 24), ("NC", 5)])
def test_tau00_full_size_against_stored_oracle_values(lt, h, key, item, panel_cluster):
    """Element-wise parity at full size where the oracle needs minutes to an hour per item: tau00 of single items of
    the largest workloads (H item 0 is the worst-conditioned matrix of all configs, cond_1 ~ 1.6e6; NC is the paper's
    rank-12450 NiAu shape) against values the oracle wrote into tests/golden/ (tests/golden/make_golden_full_size.py:
    oracle.assemble_M + FP64 LU with long-double iterative refinement; nothing there comes from the CUDA path).
    panel_cluster = 0: what a one-matrix call gets by default, the CLUSTER panel kernel on panels of >= 2048 rows;
    panel_cluster = 1: the ONE-CTA panel kernels that every batch of three or more matrices runs on -- the kernels
    bench.py times H / N / NC on: k_panel_reg<512,20,1,0> (H, N: 5121-10240 rows), <512,32,1,0> (NC: > 10240 rows),
    <512,10,2,2> (C), <512,5,4,4> (P), and the shorter instances as the panels shrink."""
    n, k, ref = read_golden(key, item)
    batch = sl.make_batch(key).select([item])
    assert batch.cfg.n == n and batch.cfg.k == k
    h.set("panel_cluster", panel_cluster)
    tau, info, _ = lt.tau00_from_liz_batch(h, batch)
    assert not info.any()
    print(f"full-size parity {key}_{item} panel_cluster={panel_cluster}: rel. Frobenius {relF(tau[0], ref):.2e}")
    check_tau(tau[0], ref, TAU_TOL, (key, item, panel_cluster))


@pytest.mark.parametrize("items", [[0, 5, 11, 17, 23], [0, 11, 23]])
def test_tau00_high_l_small_batches_through_a_default_handle(lt, h, items):
    """Workload H (6750 x 6750, spin-canted, l_max = 4) in batches of more than two matrices through a DEFAULT handle --
    lock-step schedule, look-ahead.  Five matrices: the launch shape `bench.py --workload H` times, tall panels on the
    one-CTA kernel k_panel_reg<512,20,1,0> (the scheduler uses it from five matrices on).  Three matrices: the scheduler's
    pick for three or four tall matrices, a cluster of two CTAs per panel while it is >= 4096 rows, the one-CTA kernel
    below.  Checked: the residual of the central block column on every item, tau00 equal to that column's central block,
    and the two items with stored oracle values (0: worst-conditioned of all configs; 23) element by element."""
    batch = sl.make_batch("H").select(items)
    cfg = batch.cfg
    n, k, B = cfg.n, cfg.k, len(items)
    M, _, _ = gpu_M(lt, h, batch)
    X, info = lt.lsms_solve_central_column_batched(h, M, cfg.n_sites, cfg.kmax, True, B)
    torch.cuda.synchronize()
    assert lt.lsms_last_schedule(h) == 0 and h.get("panel_cluster") == 0 and not info.cpu().numpy().any()
    res = device_residuals(M, X, n, k)
    assert float(res.max()) < RES_TOL, res
    tau, info2 = lt.lsms_tau00_batched(h, M, cfg.n_sites, cfg.kmax, True, B)                  # overwrites M
    torch.cuda.synchronize()
    assert lt.lsms_last_schedule(h) == 0 and not info2.cpu().numpy().any()
    assert float((X[:, :, n - k:] - tau).abs().max()) == 0.0
    tau = tau.cpu().numpy().transpose(0, 2, 1)
    for i, item in ((0, 0), (B - 1, 23)):
        _, _, ref = read_golden("H", item)
        print(f"H item {item} in a batch of {B}: rel. Frobenius {relF(tau[i], ref):.2e}")
        check_tau(tau[i], ref, TAU_TOL, ("H batch", B, item))


@pytest.mark.parametrize("key,item", [("N", 23), ("NC", 0)])
def test_tau00_paper_niau_shapes_properties(lt, h, key, item):
    """the paper's own NiAu ranks 6225 and 12450 (N_LIZ = 249, l_max = 4).  Same
    property checks as the high-l case: assembled M equals the oracle's M block by block, the central block column
    solves M X = E to <= 1e-12, and tau00 is the central block of X (checked against lsms_tau00_batched itself)."""
    batch = sl.make_batch(key).select([item])
    cfg = batch.cfg
    assert cfg.n == {"N": 6225, "NC": 12450}[key]
    M, _, _ = gpu_M(lt, h, batch)
    X, info = lt.lsms_solve_central_column_batched(h, M, cfg.n_sites, cfg.kmax, cfg.spin_canted, 1)
    torch.cuda.synchronize()
    assert not info.cpu().numpy().any()
    Mo = oracle_M(batch, 0)
    assert block_rel_err(M[0].cpu().numpy().T, Mo, cfg.k) < ASM_TOL
    Xh = X[0].cpu().numpy().T
    assert residual(Mo, Xh, cfg.k) < RES_TOL
    tau, info2 = lt.lsms_tau00_batched(h, M, cfg.n_sites, cfg.kmax, cfg.spin_canted, 1)      # overwrites M
    torch.cuda.synchronize()
    assert not info2.cpu().numpy().any()
    assert relF(tau[0].cpu().numpy().T, Xh[cfg.n - cfg.k:, :]) < 1e-12


# ------------------------------------------------------------------ direct input to lsms_tau00_batched

def lapack_tau00(A, k):
    """A [col, row] as stored -> central block of the inverse by LAPACK"""
    n = A.shape[0]
    return np.linalg.inv(A.T)[n - k:, n - k:]


@pytest.mark.parametrize("small", [0, 1, 2, 3, 5, 7])
@pytest.mark.parametrize("n_sites,kmax,canted", [(7, 9, False), (37, 1, False), (1, 16, False), (2, 4, True),
                                                  (33, 4, False), (5, 25, True), (129, 1, False), (23, 9, False), (150, 9, False),
                                                  (13, 16, False), (27, 4, True), (2, 25, True), (43, 4, False)])
def test_random_matrices_vs_lapack(lt, h, n_sites, kmax, canted, small):
    """Dense random matrices (strong pivoting) of ragged shapes through the lock-step schedule (small = 1), the
    small-matrix mode through L2 with the cluster size chosen by the scheduler (2), one CTA per matrix (3) and a 4-CTA
    cluster (5), the on-chip small-matrix mode (7: matrix in the distributed shared memory of a 1/2/4-CTA cluster, shapes
    with ragged last column blocks, ragged last panels and k up to 100) and the scheduler's own choice (0)."""
    k = kmax * (2 if canted else 1)
    n = n_sites * k
    h.set("small_mode", small)
    A = sl.random_dense_matrices(5, n, seed=100 + n)
    M = torch.from_numpy(A).cuda()
    tau, info = lt.lsms_tau00_batched(h, M, n_sites, kmax, canted, 5)
    torch.cuda.synchronize()
    sched = lt.lsms_last_schedule(h)
    if small in (0, 7):            # on chip (100 + cluster size) when the matrix fits the shared memory of <= 8 SMs
        if n <= 216:
            assert sched == 101 if n <= 112 else sched > 101
        if n > 256:
            assert sched == 0
    else:
        assert sched == {1: 0, 2: 4 if n <= 212 else 8, 3: 1, 5: 4}[small]
    tau = tau.cpu().numpy().transpose(0, 2, 1)
    assert not info.cpu().numpy().any()
    for b in range(5):
        check_tau(tau[b], lapack_tau00(A[b], k), 1e-10 if n > 1000 else 1e-11, (n, b))


@pytest.mark.parametrize("small", [0, 1, 2, 3, 4, 6, 7])
def test_needs_pivoting_and_singular_info(lt, h, small):
    # zero on the leading diagonal: fails without row interchanges
    n_sites, kmax = 6, 4
    n = 24
    h.set("small_mode", small)
    rng = np.random.default_rng(3)
    A = rng.standard_normal((3, n, n)) + 1j * rng.standard_normal((3, n, n))
    for j in range(n):
        A[0, j, j] = 0.0                       # column-major storage: [b, col, row]
    A[2, 5, :] = 0.0                           # column 5 identically zero -> exact zero pivot at step 6
    M = torch.from_numpy(np.ascontiguousarray(A)).cuda()
    tau, info = lt.lsms_tau00_batched(h, M, n_sites, kmax, False, 3)
    torch.cuda.synchronize()
    info = info.cpu().numpy()
    tau = tau.cpu().numpy().transpose(0, 2, 1)
    assert info[0] == 0 and info[1] == 0
    for b in (0, 1):
        check_tau(tau[b], lapack_tau00(A[b], 4), 1e-11)
    assert info[2] == 6
    # singular central block: the failure is found by the final k x k inverse, step n-k+1 .. n
    A2 = rng.standard_normal((1, n, n)) + 1j * rng.standard_normal((1, n, n))
    A2[0, n - 1, :] = 0.0
    _, info = lt.lsms_tau00_batched(h, torch.from_numpy(A2).cuda(), n_sites, kmax, False, 1)
    torch.cuda.synchronize()
    assert n - 4 < int(info.cpu().numpy()[0]) <= n


@pytest.mark.parametrize("small", [1, 3, 5])
def test_blocking_parameters_do_not_change_the_result(lt, h, small):
    batch = sl.make_batch("T").select([0, 9])
    ref, _ = oracle.tau00_batched(batch, "long double")
    h.set("small_mode", small)
    for nb, ib in ((16, 4), (32, 16), (48, 12), (96, 16), (64, 7), (0, 0)):
        h.set("nb_outer", nb).set("ib_inner", ib)
        tau, info, _ = lt.tau00_from_liz_batch(h, batch)
        assert not info.any()
        for b in range(2):
            check_tau(tau[b], ref[b], 1e-12, (nb, ib, b))


def test_lookahead_on_and_off_give_identical_results(lt, h):
    """The look-ahead split of the Schur update only re-orders independent tiles: bitwise equal tau00."""
    batch = sl.make_batch("M").select([3, 300])
    h.set("small_mode", 1)
    h.set("lookahead", 0)
    tau0, info0, _ = lt.tau00_from_liz_batch(h, batch)
    h.set("lookahead", 1)
    tau1, info1, _ = lt.tau00_from_liz_batch(h, batch)
    assert not info0.any() and not info1.any()
    assert np.array_equal(tau0, tau1)


@pytest.mark.parametrize("threads", [0, 1, 2])
def test_panel_kernel_variants_match_oracle(lt, h, threads):
    """The three K2 footprints (LSMS_OPT_PANEL_THREADS: 0 = 256 threads throughout, 1 = 512 threads on tall panels,
    2 = 128 threads up to 1024 rows) against the oracle on a tiny LIZ, ragged random matrices (w and sub-panel tails), a
    mid LIZ (several row chunks) and single items of P and C with stored oracle values, one-CTA panel kernel forced.
    Which k_panel_reg instances that reaches (panel height m = n - c0 shrinks through the shorter ones):
      threads = 2: <128,1,4,4> <128,2,4,4> (T, 207, 164 rows), <128,4,4,4> <128,8,2,3> (M: 880 rows), the 256-thread ones above
      threads = 0: <256,1,4,4> <256,2,4,4> <256,5,4,4> (<= 1280 rows), <256,10,2,2> (P: 2160), <256,20,1,0> (C: 4320)
      threads = 1: the same up to 1280 rows, <512,5,4,4> (P), <512,10,2,2> (C); the taller <512,20,1,0> / <512,32,1,0> are
                   reached by test_tau00_full_size_against_stored_oracle_values[panel_cluster=1] and the H batch of three."""
    h.set("panel_threads", threads).set("small_mode", 1).set("panel_cluster", 1)
    for key, item in (("P", 24), ("C", 24)):
        _, _, gold = read_golden(key, item)
        t, i, _ = lt.tau00_from_liz_batch(h, sl.make_batch(key).select([item]))
        assert not i.any()
        check_tau(t[0], gold, TAU_TOL, (key, item, threads))
    batch = sl.make_batch("T").select([0, 17, 31])
    ref, _ = oracle.tau00_batched(batch, "long double")
    tau, info, _ = lt.tau00_from_liz_batch(h, batch)
    assert not info.any()
    for b in range(3):
        check_tau(tau[b], ref[b], 1e-12)
    for n_sites, kmax in ((23, 9), (41, 4), (150, 9)):
        n = n_sites * kmax
        A = sl.random_dense_matrices(2, n, seed=700 + n)             # column-major storage: [b, col, row]
        tau, info = lt.lsms_tau00_batched(h, torch.from_numpy(A).cuda(), n_sites, kmax, False, 2)
        torch.cuda.synchronize()
        assert not info.cpu().numpy().any()
        tau = tau.cpu().numpy().transpose(0, 2, 1)
        for b in range(2):
            check_tau(tau[b], lapack_tau00(A[b], kmax), 1e-10)
    mid = sl.make_batch("M").select([5, 400])
    refm, _ = oracle.tau00_batched(mid, "long double")
    taum, infom, _ = lt.tau00_from_liz_batch(h, mid)
    assert not infom.any()
    for b in range(2):
        check_tau(taum[b], refm[b], 1e-10)


@pytest.mark.parametrize("cl", [2, 4, 8])
def test_panel_cluster_kernel_matches_one_cta_kernel_and_oracle(lt, h, cl):
    """K2 with a cluster of cl CTAs per matrix against the one-CTA kernel (the two search pivots with different
    tie-breaking among entries of nearly equal magnitude -- LIZ matrices are full of them -- so they agree to rounding,
    not bit for bit), and against the oracle / LAPACK on a tiny LIZ, ragged random matrices (rows not a multiple of the
    cluster's thread count, sub-panel tails) and a singular matrix (info)."""
    h.set("small_mode", 1)
    batch = sl.make_batch("T").select([0, 31])
    ref, _ = oracle.tau00_batched(batch, "long double")
    h.set("panel_cluster", 1)
    tau1, info1, _ = lt.tau00_from_liz_batch(h, batch)
    h.set("panel_cluster", cl)
    tau, info, _ = lt.tau00_from_liz_batch(h, batch)
    assert not info.any() and not info1.any()
    for b in range(2):
        check_tau(tau[b], tau1[b], 1e-12)
        check_tau(tau[b], ref[b], 1e-12)
    for n_sites, kmax in ((23, 9), (150, 9), (131, 16)):
        n = n_sites * kmax
        A = sl.random_dense_matrices(2, n, seed=900 + n)             # column-major storage: [b, col, row]
        h.set("panel_cluster", 1)
        t1, i1 = lt.lsms_tau00_batched(h, torch.from_numpy(A).cuda(), n_sites, kmax, False, 2)
        h.set("panel_cluster", cl)
        t2, i2 = lt.lsms_tau00_batched(h, torch.from_numpy(A).cuda(), n_sites, kmax, False, 2)
        torch.cuda.synchronize()
        assert not i1.cpu().numpy().any() and not i2.cpu().numpy().any()
        t1 = t1.cpu().numpy().transpose(0, 2, 1)
        t2 = t2.cpu().numpy().transpose(0, 2, 1)
        for b in range(2):
            check_tau(t2[b], t1[b], 1e-10)
            check_tau(t2[b], lapack_tau00(A[b], kmax), 1e-10)
    A = sl.random_dense_matrices(1, 24, seed=3)
    A[0, 5, :] = 0.0                           # column 5 identically zero -> exact zero pivot at step 6
    _, i3 = lt.lsms_tau00_batched(h, torch.from_numpy(A).cuda(), 6, 4, False, 1)
    torch.cuda.synchronize()
    assert int(i3.cpu().numpy()[0]) == 6


def test_batch_groups_give_identical_results(lt, h):
    """Batch groups run the same per-item elimination on separate streams: bitwise equal tau00 for every
    group count, including counts that do not divide the batch and exceed it."""
    batch = sl.make_batch("T").select(list(range(11)))
    ref, _ = oracle.tau00_batched(batch, "long double")
    h.set("small_mode", 1)
    out = []
    for g in (1, 2, 3, 8):
        h.set("groups", g)
        tau, info, _ = lt.tau00_from_liz_batch(h, batch)
        assert not info.any()
        out.append(tau)
    small = sl.make_batch("T").select([0, 5, 9])
    tau_s, info_s, _ = lt.tau00_from_liz_batch(h, small)
    assert not info_s.any()
    for tau in out[1:]:
        assert np.array_equal(out[0], tau)
    for b in range(11):
        check_tau(out[0][b], ref[b], TAU_TOL)
    assert np.array_equal(tau_s, out[0][[0, 5, 9]])


# ------------------------------------------------------------------ the batch scheduler's small-matrix mode (a7)

def test_small_mode_is_chosen_for_the_small_configs_and_matches_the_oracle(lt, h):
    """SURVEY 8(a) a7 / north_star "packs small LIZ matrices several per SM": with default options the scheduler
    runs T (208^2 x 32) in the one-launch small-matrix mode and larger matrices in lock-step; every cluster size gives
    tau00 within the bar of the oracle on all 32 T items, the launch count is that of one elimination kernel, and the
    general one-launch kernel (on request) matches the oracle on mid-size matrices."""
    batch = sl.make_batch("T")
    ref, _ = oracle.tau00_batched(batch, "long double")
    tau, info, _ = lt.tau00_from_liz_batch(h, batch)
    assert not info.any()
    assert lt.lsms_last_schedule(h) == 104 and lt.lsms_last_launch_count(h) == 1     # on chip, 4 SMs per matrix
    for b in range(32):
        check_tau(tau[b], ref[b], 1e-12, ("T default", b))
    for sm, cl in ((2, None), (3, 1), (4, 2), (5, 4), (6, 8), (7, 104)):
        h.set("small_mode", sm)
        tau, info, _ = lt.tau00_from_liz_batch(h, batch)
        assert not info.any()
        if cl:
            assert lt.lsms_last_schedule(h) == cl
        for b in range(32):
            check_tau(tau[b], ref[b], 1e-12, ("T", sm, b))
    h.set("small_mode", 2)
    mid = sl.make_batch("M").select(list(range(0, 512, 37)))
    refm, _ = oracle.tau00_batched(mid, "long double")
    taum, infom, _ = lt.tau00_from_liz_batch(h, mid)
    assert not infom.any() and lt.lsms_last_schedule(h) >= 1
    h.set("small_mode", 0)
    for b in range(mid.batch):
        check_tau(taum[b], refm[b], TAU_TOL, ("M", b))
    big = sl.make_batch("P").select([0])
    _, infob, _ = lt.tau00_from_liz_batch(h, big)
    assert not infob.any() and lt.lsms_last_schedule(h) == 0


def test_scheduler_leaves_the_on_chip_mode_when_the_batch_needs_many_waves_of_clusters(lt, h):
    """The on-chip kernel holds a cluster of SMs per matrix for the whole elimination: by default it is used while the
    batch needs at most ~3.5 waves of clusters (here 208^2: 4 SMs each, <= 129 matrices on 148 SMs) and the lock-step
    schedule beyond; forced (small_mode = 7) it runs any batch, wave after wave, with the same results."""
    n_sites, kmax, B = 13, 16, 160
    A = sl.random_dense_matrices(B, n_sites * kmax, seed=4242)
    tau_ls, info = lt.lsms_tau00_batched(h, torch.from_numpy(A).cuda(), n_sites, kmax, False, B)
    torch.cuda.synchronize()
    assert lt.lsms_last_schedule(h) == 0 and not info.cpu().numpy().any()
    tau_few, info = lt.lsms_tau00_batched(h, torch.from_numpy(A[:100]).cuda(), n_sites, kmax, False, 100)
    torch.cuda.synchronize()
    assert lt.lsms_last_schedule(h) == 104 and not info.cpu().numpy().any()
    h.set("small_mode", 7)
    tau_oc, info = lt.lsms_tau00_batched(h, torch.from_numpy(A).cuda(), n_sites, kmax, False, B)
    torch.cuda.synchronize()
    assert lt.lsms_last_schedule(h) == 104 and not info.cpu().numpy().any()
    tau_ls, tau_few, tau_oc = (t.cpu().numpy().transpose(0, 2, 1) for t in (tau_ls, tau_few, tau_oc))
    assert np.array_equal(tau_few, tau_oc[:100])                 # the same kernel on the same matrices, whatever the batch
    for b in range(0, B, 7):
        check_tau(tau_oc[b], tau_ls[b], 1e-11, ("on chip vs lock-step", b))
        check_tau(tau_oc[b], lapack_tau00(A[b], kmax), 1e-11, ("on chip vs LAPACK", b))


def test_cluster_capacity_is_known_to_the_scheduler(lt, h):
    """The cluster kernels are only scheduled where the device (or the SM partition this process has) can hold such a
    cluster: the capacities asked at bind time are plausible on a whole B200 (148 SMs; one CTA per SM for the on-chip and
    the tall-panel cluster kernels, so at most 148 / cl clusters) and non-zero for every cluster size the scheduler uses."""
    for cl in (1, 2, 4, 8):
        res, fus = lt.lsms_max_active_clusters(h, 0, cl), lt.lsms_max_active_clusters(h, 1, cl)
        assert 1 <= res <= 148 // cl, (cl, res)
        assert 1 <= fus <= 4 * 148 // cl, (cl, fus)
        if cl > 1:
            pc = lt.lsms_max_active_clusters(h, 2, cl)
            assert 1 <= pc <= 148 // cl, (cl, pc)
    assert lt.lsms_max_active_clusters(h, 2, 1) == 0
    assert lt.lsms_max_active_clusters(h, 0, 4) >= 30        # workload T: 32 clusters of 4 in one wave


def test_on_chip_mode_repeated_launches_are_bitwise_reproducible(lt, h):
    """The on-chip kernel synchronises its CTAs with flags, mbarriers and a polling "shipper" warp instead of cluster
    barriers: many launches in a row, batches of one wave and of several, cluster sizes 1 / 2 / 4 / 8 -- every launch
    must return, and return the same bits (the schedule inside the cluster must not leak into the arithmetic)."""
    h.set("small_mode", 7)
    for n_sites, kmax, canted, B in ((13, 16, False, 32), (13, 16, False, 150), (7, 9, False, 64), (33, 4, False, 40),
                                     (27, 4, True, 20), (2, 25, True, 9), (16, 1, False, 300)):
        k = kmax * (2 if canted else 1)
        A = sl.random_dense_matrices(B, n_sites * k, seed=77 + n_sites)
        M0 = torch.from_numpy(A).cuda()
        first = None
        for rep in range(25):
            tau, info = lt.lsms_tau00_batched(h, M0.clone(), n_sites, kmax, canted, B)
            if first is None:
                first = tau.clone()
            else:
                assert torch.equal(torch.view_as_real(tau), torch.view_as_real(first)), (n_sites, kmax, rep)
        torch.cuda.synchronize()
        assert lt.lsms_last_schedule(h) > 100 and not info.cpu().numpy().any()
        t = first.cpu().numpy().transpose(0, 2, 1)
        for b in range(0, B, max(1, B // 5)):
            check_tau(t[b], lapack_tau00(A[b], k), 1e-11, (n_sites, kmax, b))


# ------------------------------------------------------------------ boundary: re-entrancy and input validation

def test_two_host_threads_two_handles_two_streams(lt):
    """SURVEY 8(b) "re-entrant on different streams": two host threads, each with its own handle (different blockings
    and schedules), its own stream and its own batch, run lsms_tau00_batched concurrently; the results are
    bit-identical to the same calls made one after the other."""
    import threading
    jobs = [dict(items=list(range(0, 16)), opts=dict(nb_outer=32, ib_inner=8, small_mode=1, groups=2)),
            dict(items=list(range(16, 32)), opts=dict(nb_outer=64, ib_inner=16, small_mode=1, groups=3))]
    Ms = []
    h0 = lt.lsms_create()
    for j in jobs:
        M, _, _ = gpu_M(lt, h0, sl.make_batch("M").select(j["items"]))
        Ms.append(M)
    torch.cuda.synchronize()
    cfg = sl.CONFIGS["M"]

    def run(j, M, out, stream):
        hd = lt.lsms_create(**j["opts"])
        with torch.cuda.stream(stream):
            for _ in range(3):                                # several calls back to back keep both threads busy
                tau, info = lt.lsms_tau00_batched(hd, M.clone(), cfg.n_sites, cfg.kmax, False, len(j["items"]), stream=stream)
        stream.synchronize()
        out.append((tau.cpu().numpy(), info.cpu().numpy()))
        hd.destroy()

    serial = [[], []]
    for i, j in enumerate(jobs):
        run(j, Ms[i], serial[i], torch.cuda.Stream())
    conc = [[], []]
    threads = [threading.Thread(target=run, args=(j, Ms[i], conc[i], torch.cuda.Stream())) for i, j in enumerate(jobs)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    for i in range(2):
        assert not serial[i][0][1].any() and not conc[i][0][1].any()
        assert np.array_equal(serial[i][0][0], conc[i][0][0])
    h0.destroy()


def test_calls_on_a_side_stream_with_buffers_left_to_the_binding(lt, h):
    """Every call takes the stream it runs on.  With outputs and workspace omitted the binding allocates them with that
    stream current, so the caching allocator cannot hand the dropped workspace to other work while the kernels still use
    it: the whole path on a side stream, repeated with allocator churn on the default stream, gives the bits of the
    default-stream run."""
    batch = sl.make_batch("T")
    cfg, B = batch.cfg, batch.batch
    delta, species, z, pos, mom = lt.device_inputs(batch)
    ref, info, _ = lt.tau00_from_liz_batch(h, batch)
    assert not info.any()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    for rep in range(5):
        tinv, kappa, _ = lt.lsms_tinv_from_phase_shifts(h, delta, species, z, cfg.lmax, cfg.n_sites, False, 2, B, stream=side)
        M, _ = lt.lsms_build_M_batched(h, tinv, pos, None, kappa, cfg.lmax, cfg.n_sites, False, B, stream=side)
        tau, info = lt.lsms_tau00_batched(h, M, cfg.n_sites, cfg.kmax, False, B, stream=side)
        junk = [torch.full((1 << 18,), float(rep), device="cuda") for _ in range(8)]      # default-stream allocations meanwhile
        del junk
        side.synchronize()
        assert tau.is_cuda and not info.cpu().numpy().any()
        assert np.array_equal(tau.cpu().numpy().transpose(0, 2, 1), ref), rep


def test_illegal_input_values_are_flagged_per_item(lt, h):
    """Reading A4: Im z < 0 / Im kappa < 0 and non-finite inputs are rejected per item through info[],
    on the device and without a sync; legal items of the same batch are unaffected."""
    batch = sl.make_batch("T").select([0, 1, 2, 3, 4])
    cfg = batch.cfg
    ref, _ = oracle.tau00_batched(batch, "long double")
    delta, species, z, pos, mom = lt.device_inputs(batch)
    z = z.clone(); species = species.clone()
    z[1] = complex(0.3, -0.1)                                   # wrong half plane
    z[3] = complex(float("nan"), 0.0)
    species[4, 7] = 2                                           # only species 0 and 1 exist
    tinv, kappa, info0 = lt.lsms_tinv_from_phase_shifts(h, delta, species, z, cfg.lmax, cfg.n_sites, False, 2, 5)
    assert info0.cpu().numpy().tolist() == [0, -4, 0, -4, -2]
    kappa2 = kappa.clone()
    kappa2[1] = complex(0.5, -0.2); kappa2[3] = complex(0.5, 0.2); kappa2[4] = complex(float("inf"), 0.0)
    tinv2 = torch.nan_to_num(tinv, nan=1.0)
    M, info1 = lt.lsms_build_M_batched(h, tinv2, pos, None, kappa2, cfg.lmax, cfg.n_sites, False, 5)
    assert info1.cpu().numpy().tolist() == [0, -5, 0, 0, -5]
    assert bool(torch.isnan(torch.view_as_real(M[1])).all()) and bool(torch.isnan(torch.view_as_real(M[4])).all())
    assert bool(torch.isfinite(torch.view_as_real(M[0])).all()) and bool(torch.isfinite(torch.view_as_real(M[3])).all())
    tau, info2 = lt.lsms_tau00_batched(h, M, cfg.n_sites, cfg.kmax, False, 5)
    info2 = info2.cpu().numpy()
    assert info2[0] == 0 and info2[2] == 0 and info2[1] > 0 and info2[4] > 0       # NaN matrices fail at their first pivot
    tau = tau.cpu().numpy().transpose(0, 2, 1)
    for b in (0, 2):
        check_tau(tau[b], ref[b], 1e-12)
    # a non-finite phase shift
    d2 = delta.clone(); d2[1, 0, 2] = complex(float("inf"), 0.0)
    _, _, info3 = lt.lsms_tinv_from_phase_shifts(h, d2, lt.device_inputs(batch)[1], lt.device_inputs(batch)[2], cfg.lmax, cfg.n_sites, False, 2, 5)
    assert (info3.cpu().numpy() == -1).all()                     # every LIZ of this batch contains species 1
    # the host entry point reports the first code of the three stages
    hc = lt.HostCall(h, cfg.n_sites, cfg.lmax, False, 2, 5)
    hc.load(batch)
    hc.z[1] = complex(0.3, -0.1)
    _, info_h = hc.run()
    info_h = info_h.numpy()
    assert info_h[1] == -4 and not info_h[[0, 2, 3, 4]].any()


def test_schur_update_alone_matches_numpy(lt, h):
    """K4 in isolation: C -= A B on ragged shapes (several tiles + tails in M, N and K; K of 1..6 chunks, so both the
    one-stage and the two-stage ring are exercised)."""
    if True:
        for n, c0, kk, nb in ((333, 10, 64, 2), (200, 0, 37, 2), (130, 3, 16, 2), (97, 40, 5, 2), (700, 20, 96, 3), (450, 7, 48, 5),
                              (1100, 0, 64, 1)):
            A = sl.random_dense_matrices(nb, n, seed=n)
            M = torch.from_numpy(A).cuda()
            lt.lsms_schur_update_batched(h, M, n, c0, kk, nb)
            torch.cuda.synchronize()
            out = M.cpu().numpy().transpose(0, 2, 1)
            for b in range(nb):
                ref = A[b].T.copy()
                r0 = c0 + kk
                ref[r0:, r0:] -= ref[r0:, c0:r0] @ ref[c0:r0, r0:]
                assert np.max(np.abs(out[b] - ref)) < 1e-12 * np.abs(ref).max() * kk


# ------------------------------------------------------------------ contour reduction

def test_contour_sum_matches_oracle(lt, h):
    """sum_q w_q tau00_{a,q} on the device vs the oracle's loop: the real tau00 of two tiny-LIZ atoms on the full
    32-point contour, plus ragged shapes (k*k not a multiple of the block, one energy, many atoms)."""
    cfg = sl.custom_config(13, 3, False, n_atoms=2, n_energies=32, index=0)
    batch = sl.make_batch(cfg)
    tau, info, _ = lt.tau00_from_liz_batch(h, batch)
    assert not info.any()
    w = sl.contour_weights("semicircle", 32)
    ref = oracle.contour_sum(tau.reshape(2, 32, cfg.k, cfg.k), w)
    tau_d = torch.from_numpy(np.ascontiguousarray(tau)).cuda()
    out = lt.lsms_contour_sum_batched(h, tau_d, torch.from_numpy(w).cuda(), 2, 32, cfg.k)
    torch.cuda.synchronize()
    assert relF(out.cpu().numpy(), ref) < 1e-14
    rng = np.random.default_rng(11)
    for na, ne, k in ((1, 1, 1), (5, 24, 50), (300, 3, 7), (2, 33, 13)):
        t = rng.standard_normal((na, ne, k, k)) + 1j * rng.standard_normal((na, ne, k, k))
        ww = rng.standard_normal(ne) + 1j * rng.standard_normal(ne)
        out = lt.lsms_contour_sum_batched(h, torch.from_numpy(t).cuda(), torch.from_numpy(ww).cuda(), na, ne, k)
        torch.cuda.synchronize()
        ref = oracle.contour_sum(t, ww)
        assert np.max(np.abs(out.cpu().numpy() - ref)) < 1e-13 * np.sqrt(ne) * np.abs(t).max() * np.abs(ww).max()


# ------------------------------------------------------------------ end-to-end host entry point

def test_host_entry_point_matches_device_path(lt, h):
    batch = sl.make_batch("T")
    cfg = batch.cfg
    hc = lt.HostCall(h, cfg.n_sites, cfg.lmax, cfg.spin_canted, 2, batch.batch)
    hc.load(batch)
    tau_h, info_h = hc.run()
    launches = lt.lsms_last_launch_count(h)
    tau_d, info_d, _ = lt.tau00_from_liz_batch(h, batch)
    assert not info_h.numpy().any()
    assert np.array_equal(tau_h.numpy().transpose(0, 2, 1), tau_d)
    assert hc.h2d_bytes == batch.delta.nbytes + batch.species.nbytes + batch.z.nbytes + batch.site_pos.nbytes
    assert hc.d2h_bytes == 32 * 16 * 16 * 16 + 32 * 4
    assert 4 <= launches <= 6           # t^-1, two tables, assembly, ONE elimination launch (small-matrix mode)
    # f3 through the host call: (atoms x energies) on one lattice -> shared-g0 assembly, same bits
    cfg2 = sl.custom_config(13, 2, True, n_atoms=3, n_energies=4)
    b2 = sl.make_batch(cfg2)
    out = []
    for ne in (0, cfg2.n_energies):
        hc2 = lt.HostCall(h, cfg2.n_sites, cfg2.lmax, True, 2, b2.batch, n_energies=ne)
        hc2.load(b2)
        t, i = hc2.run()
        assert not i.numpy().any()
        out.append(t.numpy().copy())
    assert np.array_equal(out[0], out[1])


# ------------------------------------------------------------------ f2: the N > 1 path of bench.py on a device

def test_bench_two_ranks_share_one_gpu_and_gather_in_global_batch_order(lt, tmp_path):
    """SURVEY 8(e)/(f) f2 (ranks spread over GPUs, each with its own atoms): bench.py's N > 1 branch --
    process group, atoms sharded per rank, barrier + MAX-over-ranks timing, gather of the k x k blocks after the timed
    region -- executed with real kernels.  This box has one GPU, so both ranks use cuda:0 (they never wait for each
    other's kernels: there is no data-path collective) and the three small collectives go through gloo, NCCL refusing two
    ranks on one device.  Checked: exit code, n_gpus, and all 2 x 32 gathered blocks against the oracle on the GLOBAL
    batch (atom 0's energies, then atom 1's), i.e. every rank computed its own atoms and the gather kept the order."""
    import json
    import socket
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    out = str(tmp_path / "gathered.npy")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), "bench.py", "--gpus", "2", "--dist-backend", "gloo", "--all-ranks-on-device", "0",
           "--workload", "T", "--steps", "2", "--warmup", "3", "--no-cpu-baseline", "--save-gathered", out]
    r = subprocess.run(cmd, cwd=root, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, (r.stdout[-1500:], r.stderr[-3000:])
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                    # rank 0 alone prints
    line = json.loads(lines[0])
    cfg = sl.CONFIGS["T"]
    assert line["n_gpus"] == 2 and line["scaling"] == "weak" and line["parity"]["ok"]
    assert abs(line["value"] - 2 * cfg.batch / (line["ms_per_step"] * 1e-3)) < 1e-6 * line["value"]
    full = np.load(out).transpose(0, 2, 1)                    # stored column-major -> [b, row, col]
    glob = sl.make_batch(cfg, n_atoms=2)
    assert full.shape == (2 * cfg.batch, cfg.k, cfg.k) and glob.batch == 2 * cfg.batch
    ref, oinfo = oracle.tau00_batched(glob, "double")
    assert not oinfo.any()
    for b in range(glob.batch):
        check_tau(full[b], ref[b], TAU_TOL, ("two ranks", b))
    assert relF(full[cfg.batch], full[0]) > 1e-3              # atom 1 is not a copy of atom 0
