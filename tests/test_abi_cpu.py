"""CPU-side checks of the C-ABI library: it loads, exports every symbol the header declares,
its host-only functions behave, and invalid arguments are rejected before any GPU work."""
import ctypes
import os
import re

import numpy as np

import oracle
import paper_2308_16317_b200 as lt

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_functions(name):
    src = open(os.path.join(ROOT, "include", name)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lsms_[a-zA-Z0-9_]+)\s*\(", src)))


def test_library_loads_and_exports_every_declared_symbol():
    """Both headers: the method's boundary (lsms_tau.h) and the measurement/debug exports (lsms_tau_diag.h)."""
    L = lt.lib()
    method, diag = header_functions("lsms_tau.h"), header_functions("lsms_tau_diag.h")
    assert len(method) >= 12 and len(diag) >= 6 and not set(method) & set(diag)
    for name in method + diag:
        assert hasattr(L, name), name
    assert set(method + diag) == set(lt.EXPORTS)
    # nothing that measures or debugs is declared in the method's header
    assert not [n for n in method if any(w in n for w in ("profile", "probe", "debug", "launch_count", "schedule", "schur_update"))]
    # the library exports nothing beyond the two headers (no process-wide knobs left)
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", lt.LIB_PATH], capture_output=True, text=True).stdout
    exported = sorted(set(re.findall(r"\b(lsms_[a-zA-Z0-9_]+)\b", out)))
    assert exported == sorted(method + diag), set(exported) ^ set(method + diag)
    assert "sm_100a" in lt.lsms_version()


def test_handle_options_and_workspace_queries():
    """Host-only part of the handle API: works without a device (a handle binds to a device on first GPU use)."""
    h = lt.lsms_create()
    assert h.get("nb_outer") == 0 and h.get("lookahead") == 1 and h.get("small_mode") == 0
    L = lt.lib()
    assert L.lsms_set_option(h.ptr, lt.LSMS_OPT_NB_OUTER, 63) == -3 and L.lsms_set_option(h.ptr, lt.LSMS_OPT_IB_INNER, 17) == -3
    assert L.lsms_set_option(h.ptr, 99, 0) == -2 and L.lsms_set_option(None, 0, 0) == -1
    assert L.lsms_set_option(h.ptr, lt.LSMS_OPT_PANEL_CLUSTER, 3) == -3 and L.lsms_set_option(h.ptr, lt.LSMS_OPT_GROUPS, 9) == -3
    assert L.lsms_set_option(h.ptr, lt.LSMS_OPT_SMALL_MODE, 8) == -3 and L.lsms_set_option(h.ptr, lt.LSMS_OPT_PANEL_THREADS, 3) == -3
    h.set("small_mode", 7).set("panel_threads", 2)                       # on-chip mode forced; quarter-SM panel kernel
    assert h.get("small_mode") == 7 and h.get("panel_threads") == 2
    h.set("small_mode", 0).set("panel_threads", 1)
    w64 = lt.lsms_workspace_bytes(h, 135, 3, False, 128)
    assert w64 >= 128 * 2160 * 4
    h.set("nb_outer", 32)
    assert lt.lsms_workspace_bytes(h, 135, 3, False, 128) < w64          # the workspace depends on the handle's NB, explicitly
    h.set("nb_outer", 0)
    assert lt.lsms_workspace_bytes(h, 0, 3, False, 1) == 0
    assert lt.lsms_workspace_bytes(h, 13, 9, False, 1) == 0
    n = 13 * 16
    assert lt.lsms_solve_workspace_bytes(h, 13, 16, False, 2) >= 2 * n * n * 16
    assert lt.lsms_host_call_scratch_bytes(h, 13, 3, False, 2, 32) >= 32 * n * n * 16
    assert lt.lsms_last_schedule(h) == -1
    h2 = lt.lsms_create(nb_outer=48)                                     # handles are independent
    assert h2.get("nb_outer") == 48 and h.get("nb_outer") == 0
    h.destroy(); h2.destroy()


def test_invalid_arguments_are_rejected_without_gpu_work():
    L = lt.lib()
    h = lt.lsms_create()
    H = h.ptr
    buf = (ctypes.c_double * 64)()
    p = ctypes.addressof(buf)
    p16 = (p + 15) // 16 * 16
    assert L.lsms_tau00_batched(None, p16, 13, 16, 0, 1, p16, p16, p16, 1 << 20, 0) == -1
    assert L.lsms_tau00_batched(H, 0, 13, 16, 0, 1, p16, p16, p16, 1 << 20, 0) == -2
    assert L.lsms_tau00_batched(H, p16 + 8, 13, 16, 0, 1, p16, p16, p16, 1 << 20, 0) == -2      # misaligned
    assert L.lsms_tau00_batched(H, p16, 0, 16, 0, 1, p16, p16, p16, 1 << 20, 0) == -3
    assert L.lsms_tau00_batched(H, p16, 13, 15, 0, 1, p16, p16, p16, 1 << 20, 0) == -4          # not a perfect square
    assert L.lsms_tau00_batched(H, p16, 13, 16, 0, 0, p16, p16, p16, 1 << 20, 0) == -6
    assert L.lsms_tau00_batched(H, p16, 13, 16, 0, 1, 0, p16, p16, 1 << 20, 0) == -7
    assert L.lsms_tau00_batched(H, p16, 13, 16, 0, 1, p16, 0, p16, 1 << 20, 0) == -8
    assert L.lsms_tau00_batched(H, p16, 13, 16, 0, 1, p16, p16, 0, 1 << 20, 0) == -9
    assert L.lsms_tau00_batched(H, p16, 13, 16, 0, 1, p16, p16, p16, 16, 0) == -10              # workspace too small
    assert L.lsms_build_M_batched(None, p16, p16, 0, p16, 3, 13, 0, 1, p16, p16, p16, 1 << 20, 0) == -1
    assert L.lsms_build_M_batched(H, 0, p16, 0, p16, 3, 13, 0, 1, p16, p16, p16, 1 << 20, 0) == -2
    assert L.lsms_build_M_batched(H, p16, p16, 0, p16, 3, 13, 1, 1, p16, p16, p16, 1 << 20, 0) == -4  # canted needs moments
    assert L.lsms_build_M_batched(H, p16, p16, 0, p16, 9, 13, 0, 1, p16, p16, p16, 1 << 20, 0) == -6
    assert L.lsms_build_M_batched(H, p16, p16, 0, p16, 3, 13, 0, 1, p16, 0, p16, 1 << 20, 0) == -11   # info
    assert L.lsms_build_M_batched(H, p16, p16, 0, p16, 3, 13, 0, 1, p16, p16, p16, 16, 0) == -13
    assert L.lsms_tinv_from_phase_shifts(H, p16, p16, p16, 3, 13, 0, 2, 1, p16, p16, 0, 0) == -12
    assert L.lsms_tau00_from_host(H, p16, p16, p16, p16, 0, 3, 13, 0, 2, 4, 5, p16, p16, p16, 1 << 20, 0, None, None) == -12
    assert L.lsms_contour_sum_batched(H, p16, p16, 1, 0, 4, p16, 0) == -5
    assert L.lsms_schur_update_batched(H, p16, 100, 90, 10, 1, 0) == -4
    assert L.lsms_destroy(None) == -1 and L.lsms_create(None) == -1
    h.destroy()


def test_panel_heights_beyond_the_kernels_are_rejected_up_front():
    """The one-CTA panel kernels cover 16384 rows; the cluster panel kernel covers 40960 rows for one or two matrices per
    call (8 CTAs) and 20480 for three or four (4 CTAs): a larger matrix is refused with its own code before anything is
    enqueued, and the workspace queries answer 0."""
    L = lt.lib()
    h = lt.lsms_create()
    buf = (ctypes.c_double * 64)()
    p16 = (ctypes.addressof(buf) + 15) // 16 * 16
    assert lt.LSMS_ERR_PANEL_TOO_TALL == -22
    assert lt.lsms_workspace_bytes(h, 1024, 3, False, 5) > 0                      # 16384 rows
    assert lt.lsms_workspace_bytes(h, 1100, 3, False, 5) == 0                     # 17600 rows, five matrices
    assert lt.lsms_workspace_bytes(h, 1100, 3, False, 4) > 0                      # ... four: clusters of 4 CTAs
    assert lt.lsms_workspace_bytes(h, 1300, 3, False, 4) == 0                     # 20800 rows: beyond 4 x 5120
    assert lt.lsms_workspace_bytes(h, 1300, 3, False, 2) > 0                      # ... two: clusters of 8 CTAs
    assert lt.lsms_workspace_bytes(h, 2600, 3, False, 1) == 0                     # 41600 rows: beyond 8 x 5120
    assert L.lsms_tau00_batched(h.ptr, p16, 1100, 16, 0, 5, p16, p16, p16, 1 << 40, 0) == -22
    assert L.lsms_solve_central_column_batched(h.ptr, p16, 1100, 16, 0, 5, p16, p16, p16, 1 << 40, 0) == -22
    assert L.lsms_tau00_from_host(h.ptr, p16, p16, p16, p16, 0, 3, 1100, 0, 2, 5, 0, p16, p16, p16, 1 << 40, 0, None, None) == -22
    h.set("panel_cluster", 1)                                                     # cluster kernel ruled out by the caller
    assert lt.lsms_workspace_bytes(h, 1100, 3, False, 1) == 0
    assert L.lsms_tau00_batched(h.ptr, p16, 1100, 16, 0, 1, p16, p16, p16, 1 << 40, 0) == -22
    assert L.lsms_set_option(h.ptr, lt.LSMS_OPT_LOOKAHEAD, 2) == -3               # 0 / 1 only
    assert L.lsms_max_active_clusters(None, 0, 4, None) == -1 and L.lsms_max_active_clusters(h.ptr, 3, 4, None) == -2
    assert L.lsms_max_active_clusters(h.ptr, 0, 3, None) == -3 and L.lsms_max_active_clusters(h.ptr, 0, 4, None) == -4
    h.destroy()


def test_closed_form_gaunt_matches_oracle_quadrature():
    """K1 tabulates Gaunt numbers from Wigner 3j symbols; the oracle integrates numerically."""
    for lmax in (3, 4):
        T = oracle.gaunt_table(lmax)
        kmax = (lmax + 1) ** 2
        worst = 0.0
        for L in range(kmax):
            l = int(np.sqrt(L)); m = L - l * (l + 1)
            for Lp in range(kmax):
                lp = int(np.sqrt(Lp)); mp = Lp - lp * (lp + 1)
                for lpp in range(0, 2 * lmax + 1):
                    mpp = mp - m
                    ref = T[L, Lp, lpp * (lpp + 1) + mpp] if abs(mpp) <= lpp else 0.0
                    worst = max(worst, abs(lt.lsms_debug_gaunt_closed_form(l, m, lp, mp, lpp) - ref))
        assert worst < 1e-14, worst
