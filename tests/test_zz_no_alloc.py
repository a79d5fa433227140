"""The allocation-free entry point, lsms_tau00_onchip_static_scratch, against the ordinary path.

Some callers of this library cannot allocate device memory when they need tau00: MPI ranks that share a GPU and sized
all their device buffers at start-up -- a cudaMalloc in their energy loop may fail and stalls the
device for every rank on it -- and host codes whose device memory is owned by another runtime.  For them the library
has one call that takes inputs and outputs only; its pivot scratch is a fixed 256 KB array inside the library.

This file is named so that pytest collects it LAST: it is the only test that touches the library's one piece of
process-wide state, and with `pytest -x` a failure here must not hide the parity tests.  It has to pass both on its own
in a fresh process (the first call does the per-device set-up) and after every other test has run.
"""
import ctypes

import numpy as np
import pytest

import synth_liz as sl

TAU_TOL = 1e-10          # the bar of tests/test_gpu_parity.py (relative Frobenius and max-element)


def _rel_errors(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b), float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


@pytest.mark.gpu
def test_static_scratch_call_matches_the_workspace_path_twice_in_a_row():
    """Two calls in a row on DIFFERENT batches (the second finds the first one's pivots in the shared array, at other
    offsets: 208-row items, then 234-row items): each must give what lsms_tau00_batched gives in on-chip mode from a
    caller-supplied workspace, within the parity tolerance, with identical info."""
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2308_16317_b200 as lt
    lt.lib()
    h = lt.lsms_create(small_mode=7)                     # the existing path: on-chip schedule, pivots in the workspace
    cases = (sl.custom_config(13, 3, False, n_energies=32, index=0),       # workload T's shape: 208 x 208 x 32
             sl.custom_config(13, 2, True, n_energies=12))                 # spin-canted, 234 x 234 x 12
    for cfg in cases:
        batch = sl.make_batch(cfg)
        B, k = batch.batch, cfg.k
        assert B * cfg.n <= lt.LSMS_STATIC_SCRATCH_WORDS
        delta, species, z, pos, mom = lt.device_inputs(batch)
        tinv, kappa, _ = lt.lsms_tinv_from_phase_shifts(h, delta, species, z, cfg.lmax, cfg.n_sites, cfg.spin_canted,
                                                        batch.delta.shape[0], B)
        M, _ = lt.lsms_build_M_batched(h, tinv, pos, mom if cfg.spin_canted else None, kappa, cfg.lmax, cfg.n_sites,
                                       cfg.spin_canted, B)
        M2 = M.clone()
        ref, ref_info = lt.lsms_tau00_batched(h, M, cfg.n_sites, cfg.kmax, cfg.spin_canted, B)
        assert lt.lsms_last_schedule(h) > 100
        # the caller's own buffers; garbage in the outputs must not matter
        tau = torch.full((B, k, k), float("nan"), dtype=torch.complex128, device="cuda")
        info = torch.full((B,), 77, dtype=torch.int32, device="cuda")
        lt.lsms_tau00_onchip_static_scratch(M2, cfg.n_sites, cfg.kmax, cfg.spin_canted, B, tau, info)
        torch.cuda.synchronize()
        assert not ref_info.cpu().numpy().any() and not info.cpu().numpy().any()
        fro, mx = _rel_errors(tau.cpu().numpy(), ref.cpu().numpy())
        assert fro < TAU_TOL and mx < TAU_TOL, (cfg.n, fro, mx)
        # the factorised matrices agree too (the kernel leaves U and the trailing block in M)
        fro_m, _ = _rel_errors(M2.cpu().numpy(), M.cpu().numpy())
        assert fro_m < TAU_TOL, (cfg.n, fro_m)
    h.destroy()


def test_static_scratch_call_rejects_sizes_beyond_its_limits_before_any_gpu_work():
    """Both limits are host-side checks in front of every CUDA call, so this runs without a device: a batch whose pivot
    vectors exceed the built-in array, a matrix too large for the on-chip kernel, and the argument codes."""
    import paper_2308_16317_b200 as lt
    L = lt.lib()
    buf = (ctypes.c_double * 64)()
    p16 = (ctypes.addressof(buf) + 15) // 16 * 16
    f = L.lsms_tau00_onchip_static_scratch
    n = 13 * 16
    fits = lt.LSMS_STATIC_SCRATCH_WORDS // n
    assert f(p16, 13, 16, 0, fits + 1, p16, p16, 0) == lt.LSMS_ERR_STATIC_SCRATCH_TOO_SMALL
    assert f(p16, 135, 16, 0, 1, p16, p16, 0) == lt.LSMS_ERR_NOT_ON_CHIP            # 2160 rows
    assert f(p16, 17, 16, 0, 1, p16, p16, 0) == lt.LSMS_ERR_NOT_ON_CHIP             # 272 rows > 256
    assert f(0, 13, 16, 0, 1, p16, p16, 0) == -1 and f(p16 + 8, 13, 16, 0, 1, p16, p16, 0) == -1
    assert f(p16, 0, 16, 0, 1, p16, p16, 0) == -2 and f(p16, 13, 15, 0, 1, p16, p16, 0) == -3
    assert f(p16, 13, 16, 0, 0, p16, p16, 0) == -5 and f(p16, 13, 16, 0, 1, 0, p16, 0) == -6
    assert f(p16, 13, 16, 0, 1, p16, 0, 0) == -7

    class FakeTensor:                       # the binding turns the two limit codes into messages that name the limit
        def data_ptr(self):
            return p16

    class FakeStream:
        cuda_stream = 0

    t = FakeTensor()
    with pytest.raises(lt.LsmsError, match="exceeds the built-in scratch of 65536 words"):
        lt.lsms_tau00_onchip_static_scratch(t, 13, 16, False, fits + 1, t, t, stream=FakeStream())
    with pytest.raises(lt.LsmsError, match="does not fit the on-chip kernel"):
        lt.lsms_tau00_onchip_static_scratch(t, 135, 16, False, 1, t, t, stream=FakeStream())
    with pytest.raises(lt.LsmsError, match="allocates nothing"):
        lt.lsms_tau00_onchip_static_scratch(t, 13, 16, False, 1, None, t, stream=FakeStream())
