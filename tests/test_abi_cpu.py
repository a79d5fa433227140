"""CPU-side checks of the C-ABI library: it loads, exports every symbol the header declares,
its host-only functions behave, and invalid arguments are rejected before any GPU work."""
import ctypes
import os
import re

import numpy as np

import oracle
import paper_2308_16317_b200 as lt

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_functions():
    src = open(os.path.join(ROOT, "include", "lsms_tau.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lsms_[a-zA-Z0-9_]+)\s*\(", src)))


def test_library_loads_and_exports_every_declared_symbol():
    L = lt.lib()
    names = header_functions()
    assert len(names) >= 12
    for name in names:
        assert hasattr(L, name), name
    assert set(names) == set(lt.EXPORTS)
    assert "sm_100a" in lt.lsms_version()


def test_workspace_queries():
    assert lt.lsms_workspace_bytes(135, 3, False, 128) >= 128 * 2160 * 4
    assert lt.lsms_workspace_bytes(0, 3, False, 1) == 0
    assert lt.lsms_workspace_bytes(13, 9, False, 1) == 0
    n = 13 * 16
    assert lt.lsms_solve_workspace_bytes(13, 16, False, 2) >= 2 * n * n * 16
    assert lt.lsms_host_call_scratch_bytes(13, 3, False, 2, 32) >= 32 * n * n * 16


def test_invalid_arguments_are_rejected_without_gpu_work():
    L = lt.lib()
    buf = (ctypes.c_double * 64)()
    p = ctypes.addressof(buf)
    p16 = (p + 15) // 16 * 16
    assert L.lsms_tau00_batched(0, 13, 16, 0, 1, p16, p16, p16, 1 << 20, 0) == -1
    assert L.lsms_tau00_batched(p16 + 8, 13, 16, 0, 1, p16, p16, p16, 1 << 20, 0) == -1      # misaligned
    assert L.lsms_tau00_batched(p16, 0, 16, 0, 1, p16, p16, p16, 1 << 20, 0) == -2
    assert L.lsms_tau00_batched(p16, 13, 15, 0, 1, p16, p16, p16, 1 << 20, 0) == -3          # not a perfect square
    assert L.lsms_tau00_batched(p16, 13, 16, 0, 0, p16, p16, p16, 1 << 20, 0) == -5
    assert L.lsms_tau00_batched(p16, 13, 16, 0, 1, 0, p16, p16, 1 << 20, 0) == -6
    assert L.lsms_tau00_batched(p16, 13, 16, 0, 1, p16, 0, p16, 1 << 20, 0) == -7
    assert L.lsms_tau00_batched(p16, 13, 16, 0, 1, p16, p16, 0, 1 << 20, 0) == -8
    assert L.lsms_tau00_batched(p16, 13, 16, 0, 1, p16, p16, p16, 16, 0) == -9               # workspace too small
    assert L.lsms_build_M_batched(0, p16, 0, p16, 3, 13, 0, 1, p16, p16, 1 << 20, 0) == -1
    assert L.lsms_build_M_batched(p16, p16, 0, p16, 3, 13, 1, 1, p16, p16, 1 << 20, 0) == -3  # canted needs moments
    assert L.lsms_build_M_batched(p16, p16, 0, p16, 9, 13, 0, 1, p16, p16, 1 << 20, 0) == -5
    assert L.lsms_build_M_batched(p16, p16, 0, p16, 3, 13, 0, 1, p16, p16, 16, 0) == -11
    assert L.lsms_set_blocking(63, 0) == -1 and L.lsms_set_blocking(64, 17) == -2 and L.lsms_set_blocking(0, 0) == 0
    assert L.lsms_schur_update_batched(p16, 100, 90, 10, 1, 0) == -3


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
