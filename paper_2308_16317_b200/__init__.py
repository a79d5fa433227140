"""Thin Python binding of liblsms_tau.so (include/lsms_tau.h, include/lsms_tau_diag.h) -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels of csrc/; PyTorch is used for device
memory and streams.  There is no CPU fallback: if the shared library is missing or a call
returns non-zero this module raises.

Every C function has a Python function of the same name taking the same arguments in the same order; the first
argument is a `Handle` (lsms_create / lsms_destroy) -- the library keeps no process-wide state.  Output buffers and
the workspace may be omitted (None), in which case they are allocated here with torch.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblsms_tau.so")
_lib = None

EXPORTS = (
    # include/lsms_tau.h -- the method
    "lsms_version", "lsms_create", "lsms_destroy", "lsms_set_option", "lsms_get_option",
    "lsms_workspace_bytes", "lsms_solve_workspace_bytes", "lsms_host_call_scratch_bytes",
    "lsms_tinv_from_phase_shifts", "lsms_build_M_batched", "lsms_build_M_shared_g0_batched", "lsms_tau00_batched",
    "lsms_solve_central_column_batched", "lsms_tau00_from_host", "lsms_contour_sum_batched",
    "lsms_tau00_onchip_static_scratch",
    # include/lsms_tau_diag.h -- measurement and debugging
    "lsms_last_launch_count", "lsms_last_schedule", "lsms_max_active_clusters", "lsms_profile_begin", "lsms_profile_end", "lsms_fp64_peak_probe",
    "lsms_schur_update_batched", "lsms_debug_gaunt_closed_form",
)

# option ids of include/lsms_tau.h
LSMS_OPT_NB_OUTER, LSMS_OPT_IB_INNER, LSMS_OPT_LOOKAHEAD, LSMS_OPT_GROUPS, LSMS_OPT_PANEL_THREADS, \
    LSMS_OPT_PANEL_CLUSTER, LSMS_OPT_ALIGN_FIRST, LSMS_OPT_SMALL_MODE = range(8)


class LsmsError(RuntimeError):
    pass


def lib() -> ctypes.CDLL:
    """Load liblsms_tau.so (built in-tree by paper_2308_16317_b200/build.py); fails loudly."""
    global _lib
    if _lib is None:
        # build.build() is a no-op when the library matches the sources (content hash); a fresh checkout or an
        # edited kernel is compiled here (nvcc cross-compiles without a GPU), under a file lock; never a fallback
        try:
            from . import build as _build
            _build.build()
        except Exception as exc:          # noqa: BLE001 - reported below
            if not os.path.exists(LIB_PATH):
                raise LsmsError(f"{LIB_PATH} is missing and `python paper_2308_16317_b200/build.py` failed: {exc} "
                                "(there is no CPU fallback)") from exc
            raise LsmsError(f"{LIB_PATH} is out of date and rebuilding it failed: {exc}") from exc
        L = ctypes.CDLL(LIB_PATH)
        vp, ci, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t
        L.lsms_version.restype = ctypes.c_char_p
        L.lsms_create.argtypes = [ctypes.POINTER(vp)]
        L.lsms_destroy.argtypes = [vp]
        L.lsms_set_option.argtypes = [vp, ci, ci]
        L.lsms_get_option.argtypes = [vp, ci, ctypes.POINTER(ci)]
        L.lsms_workspace_bytes.restype = sz
        L.lsms_workspace_bytes.argtypes = [vp, ci, ci, ci, ci]
        L.lsms_solve_workspace_bytes.restype = sz
        L.lsms_solve_workspace_bytes.argtypes = [vp, ci, ci, ci, ci]
        L.lsms_host_call_scratch_bytes.restype = sz
        L.lsms_host_call_scratch_bytes.argtypes = [vp, ci, ci, ci, ci, ci]
        L.lsms_tinv_from_phase_shifts.argtypes = [vp, vp, vp, vp, ci, ci, ci, ci, ci, vp, vp, vp, vp]
        L.lsms_build_M_batched.argtypes = [vp, vp, vp, vp, vp, ci, ci, ci, ci, vp, vp, vp, sz, vp]
        L.lsms_build_M_shared_g0_batched.argtypes = [vp, vp, vp, vp, vp, ci, ci, ci, ci, ci, vp, vp, vp, sz, vp]
        L.lsms_tau00_batched.argtypes = [vp, vp, ci, ci, ci, ci, vp, vp, vp, sz, vp]
        L.lsms_solve_central_column_batched.argtypes = [vp, vp, ci, ci, ci, ci, vp, vp, vp, sz, vp]
        L.lsms_tau00_onchip_static_scratch.argtypes = [vp, ci, ci, ci, ci, vp, vp, vp]
        L.lsms_tau00_from_host.argtypes = [vp, vp, vp, vp, vp, vp, ci, ci, ci, ci, ci, ci, vp, vp, vp, sz, vp,
                                           ctypes.POINTER(sz), ctypes.POINTER(sz)]
        L.lsms_contour_sum_batched.argtypes = [vp, vp, vp, ci, ci, ci, vp, vp]
        L.lsms_last_launch_count.argtypes = [vp]
        L.lsms_last_schedule.argtypes = [vp]
        L.lsms_max_active_clusters.argtypes = [vp, ci, ci, ctypes.POINTER(ci)]
        L.lsms_profile_begin.argtypes = [vp]
        L.lsms_profile_end.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ci), ctypes.POINTER(ctypes.c_double)]
        L.lsms_fp64_peak_probe.argtypes = [vp, ci, ci, vp, ctypes.POINTER(ctypes.c_double), vp]
        L.lsms_schur_update_batched.argtypes = [vp, vp, ci, ci, ci, ci, vp]
        L.lsms_debug_gaunt_closed_form.restype = ctypes.c_double
        L.lsms_debug_gaunt_closed_form.argtypes = [ci, ci, ci, ci, ci]
        _lib = L
    return _lib


LSMS_ERR_PANEL_TOO_TALL = -22


def _check(rc: int, what: str) -> None:
    if rc == LSMS_ERR_PANEL_TOO_TALL:
        raise LsmsError(f"{what}: the matrix has more rows than the panel kernels cover for this batch and these options "
                        "(16384; 20480 for three or four matrices per call, 40960 for one or two)")
    if rc != 0:
        raise LsmsError(f"{what} returned {rc} "
                        f"({'argument %d invalid' % -rc if rc < 0 else 'CUDA error code'})")


class Handle:
    """lsms_handle_t: scheduler options + the streams/events of the batch scheduler (include/lsms_tau.h)."""

    def __init__(self, **options):
        self._h = ctypes.c_void_p(None)
        _check(lib().lsms_create(ctypes.byref(self._h)), "lsms_create")
        for name, value in options.items():
            self.set(name, value)

    @property
    def ptr(self):
        if not self._h:
            raise LsmsError("handle was destroyed")
        return self._h

    @staticmethod
    def _opt(name) -> int:
        return name if isinstance(name, int) else globals()["LSMS_OPT_" + str(name).upper()]

    def set(self, name, value) -> "Handle":
        _check(lib().lsms_set_option(self.ptr, self._opt(name), int(value)), f"lsms_set_option({name}, {value})")
        return self

    def get(self, name) -> int:
        out = ctypes.c_int(0)
        _check(lib().lsms_get_option(self.ptr, self._opt(name), ctypes.byref(out)), f"lsms_get_option({name})")
        return out.value

    def destroy(self) -> None:
        if self._h:
            _check(lib().lsms_destroy(self._h), "lsms_destroy")
            self._h = ctypes.c_void_p(None)

    def __del__(self):
        try:
            if self._h and _lib is not None:
                _lib.lsms_destroy(self._h)
        except Exception:          # noqa: BLE001 - interpreter shutdown
            pass


def lsms_create(**options) -> Handle:
    return Handle(**options)


def lsms_destroy(handle: Handle) -> None:
    handle.destroy()


def lsms_set_option(handle: Handle, option, value) -> None:
    handle.set(option, value)


def lsms_get_option(handle: Handle, option) -> int:
    return handle.get(option)


def _stream(stream=None) -> int:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


def _ptr(t) -> int:
    return 0 if t is None else int(t.data_ptr())


def lsms_version() -> str:
    return lib().lsms_version().decode()


def lsms_workspace_bytes(handle: Handle, n_sites: int, lmax: int, spin_canted: bool, batch: int) -> int:
    return int(lib().lsms_workspace_bytes(handle.ptr, n_sites, lmax, int(bool(spin_canted)), batch))


def lsms_solve_workspace_bytes(handle: Handle, n_sites: int, kmax: int, spin_canted: bool, batch: int) -> int:
    return int(lib().lsms_solve_workspace_bytes(handle.ptr, n_sites, kmax, int(bool(spin_canted)), batch))


def lsms_host_call_scratch_bytes(handle: Handle, n_sites, lmax, spin_canted, n_species, batch) -> int:
    return int(lib().lsms_host_call_scratch_bytes(handle.ptr, n_sites, lmax, int(bool(spin_canted)), n_species, batch))


def lsms_last_launch_count(handle: Handle) -> int:
    return int(lib().lsms_last_launch_count(handle.ptr))


def lsms_last_schedule(handle: Handle) -> int:
    return int(lib().lsms_last_schedule(handle.ptr))


def lsms_max_active_clusters(handle: Handle, kernel: int, cluster_size: int) -> int:
    """kernel: 0 on-chip elimination, 1 one-launch elimination through L2, 2 cluster panel kernel."""
    out = ctypes.c_int(-1)
    _check(lib().lsms_max_active_clusters(handle.ptr, kernel, cluster_size, ctypes.byref(out)), "lsms_max_active_clusters")
    return out.value


KERNEL_CLASSES = ("K1_assemble", "K2_panel", "small_mode_lu", "K4_inner_gemm", "K4_schur_gemm", "K5_final_inverse",
                  "K3_permute_ninv", "K4_trsm_gemm")


def lsms_profile_begin(handle: Handle) -> None:
    _check(lib().lsms_profile_begin(handle.ptr), "lsms_profile_begin")


def lsms_profile_end(handle: Handle) -> dict:
    ms = (ctypes.c_double * 8)()
    cnt = (ctypes.c_int * 8)()
    fl = (ctypes.c_double * 8)()
    _check(lib().lsms_profile_end(handle.ptr, ms, cnt, fl), "lsms_profile_end")
    return {name: {"ms": ms[i], "launches": cnt[i], "flops": fl[i]} for i, name in enumerate(KERNEL_CLASSES)}


def lsms_debug_gaunt_closed_form(l, m, lp, mp, lpp) -> float:
    return float(lib().lsms_debug_gaunt_closed_form(l, m, lp, mp, lpp))


def lsms_fp64_peak_probe(handle: Handle, which: int, iters: int = 20000, sink=None, stream=None) -> float:
    import torch
    if sink is None:
        sink = torch.zeros(1, dtype=torch.float64, device="cuda")
    out = ctypes.c_double(0.0)
    _check(lib().lsms_fp64_peak_probe(handle.ptr, which, iters, _ptr(sink), ctypes.byref(out), _stream(stream)),
           "lsms_fp64_peak_probe")
    return out.value


def _empty(shape, dtype, device, stream=None):
    """Buffers this module allocates on the caller's behalf (omitted outputs, the workspace) are allocated with `stream`
    current -- the stream the library call runs on.  torch's caching allocator ties a block to the stream that was
    current when it was allocated: a workspace dropped when the (asynchronous) call returns may then only be reused by
    work ordered after the call on that same stream, never by another stream's work while the kernels still use it.
    (The scheduler's own streams are forked from and joined back into `stream` inside the call.)"""
    import torch
    if stream is None:
        return torch.empty(shape, dtype=dtype, device=device)
    with torch.cuda.stream(stream):
        return torch.empty(shape, dtype=dtype, device=device)


def _workspace(nbytes: int, device, stream=None):
    import torch
    return _empty(max(int(nbytes), 256), torch.uint8, device, stream)


def _info(batch, device, stream=None):
    import torch
    return _empty((batch,), torch.int32, device, stream)


def lsms_tinv_from_phase_shifts(handle: Handle, delta, species, z, lmax, n_sites, spin_canted, n_species, batch,
                                tinv_diag=None, kappa=None, info=None, stream=None):
    """delta c128 [n_species, n_spin, lmax+1], species i32 [batch, n_sites], z c128 [batch] (device tensors)
    -> (tinv_diag c128 [batch, n_sites, n_spin, lmax+1], kappa c128 [batch], info i32 [batch])."""
    import torch
    nspin = 2 if spin_canted else 1
    if tinv_diag is None:
        tinv_diag = _empty((batch, n_sites, nspin, lmax + 1), torch.complex128, z.device, stream)
    if kappa is None:
        kappa = _empty((batch,), torch.complex128, z.device, stream)
    if info is None:
        info = _info(batch, z.device, stream)
    _check(lib().lsms_tinv_from_phase_shifts(handle.ptr, _ptr(delta), _ptr(species), _ptr(z), lmax, n_sites,
                                             int(bool(spin_canted)), n_species, batch, _ptr(tinv_diag), _ptr(kappa),
                                             _ptr(info), _stream(stream)), "lsms_tinv_from_phase_shifts")
    return tinv_diag, kappa, info


def lsms_build_M_batched(handle: Handle, tinv_diag, site_pos, moment_dir, kappa, lmax, n_sites, spin_canted, batch,
                         M_out=None, info=None, workspace=None, stream=None):
    """-> (M_out c128 [batch, n, n], info); M_out[b, c, r] is element (row r, col c) (column-major storage)."""
    import torch
    k = (lmax + 1) ** 2 * (2 if spin_canted else 1)
    n = n_sites * k
    if M_out is None:
        M_out = _empty((batch, n, n), torch.complex128, kappa.device, stream)
    if info is None:
        info = _info(batch, kappa.device, stream)
    if workspace is None:
        workspace = _workspace(lsms_workspace_bytes(handle, n_sites, lmax, spin_canted, batch), kappa.device, stream)
    _check(lib().lsms_build_M_batched(handle.ptr, _ptr(tinv_diag), _ptr(site_pos), _ptr(moment_dir), _ptr(kappa), lmax,
                                      n_sites, int(bool(spin_canted)), batch, _ptr(M_out), _ptr(info), _ptr(workspace),
                                      workspace.numel(), _stream(stream)), "lsms_build_M_batched")
    return M_out, info


def lsms_build_M_shared_g0_batched(handle: Handle, tinv_diag, site_pos, moment_dir, kappa, lmax, n_sites, spin_canted,
                                   n_atoms, n_energies, M_out=None, info=None, workspace=None, stream=None):
    """De-duplicated assembly (one g0 per energy for all atoms); same outputs as lsms_build_M_batched."""
    import torch
    k = (lmax + 1) ** 2 * (2 if spin_canted else 1)
    n = n_sites * k
    batch = n_atoms * n_energies
    if M_out is None:
        M_out = _empty((batch, n, n), torch.complex128, kappa.device, stream)
    if info is None:
        info = _info(batch, kappa.device, stream)
    if workspace is None:
        workspace = _workspace(lsms_workspace_bytes(handle, n_sites, lmax, spin_canted, batch), kappa.device, stream)
    _check(lib().lsms_build_M_shared_g0_batched(handle.ptr, _ptr(tinv_diag), _ptr(site_pos), _ptr(moment_dir), _ptr(kappa),
                                                lmax, n_sites, int(bool(spin_canted)), n_atoms, n_energies, _ptr(M_out),
                                                _ptr(info), _ptr(workspace), workspace.numel(), _stream(stream)),
           "lsms_build_M_shared_g0_batched")
    return M_out, info


def lsms_tau00_batched(handle: Handle, M, n_sites, kmax, spin_canted, batch, tau00_out=None, info=None, workspace=None,
                       stream=None):
    """M c128 [batch, n, n] column-major, OVERWRITTEN -> (tau00 c128 [batch, k, k] with tau00[b, c, r] = element
    (row r, col c), info i32 [batch])."""
    import torch
    k = kmax * (2 if spin_canted else 1)
    lmax = int(round(kmax ** 0.5)) - 1
    if tau00_out is None:
        tau00_out = _empty((batch, k, k), torch.complex128, M.device, stream)
    if info is None:
        info = _info(batch, M.device, stream)
    if workspace is None:
        workspace = _workspace(lsms_workspace_bytes(handle, n_sites, max(lmax, 0), spin_canted, batch), M.device, stream)
    _check(lib().lsms_tau00_batched(handle.ptr, _ptr(M), n_sites, kmax, int(bool(spin_canted)), batch, _ptr(tau00_out),
                                    _ptr(info), _ptr(workspace), workspace.numel(), _stream(stream)), "lsms_tau00_batched")
    return tau00_out, info


LSMS_STATIC_SCRATCH_WORDS = 65536            # include/lsms_tau.h
LSMS_ERR_NOT_ON_CHIP, LSMS_ERR_STATIC_SCRATCH_TOO_SMALL = -20, -21


def lsms_tau00_onchip_static_scratch(M, n_sites, kmax, spin_canted, batch, tau00_out, info, stream=None):
    """tau00 of a batch of small matrices for callers that cannot allocate device memory (ranks that share a GPU and
    sized their buffers at start-up; host codes whose device memory another runtime owns): no handle, no workspace.
    The pivot scratch is a fixed 256 KB array inside the library, so batch * n <= LSMS_STATIC_SCRATCH_WORDS and the
    matrix must fit the on-chip kernel (n <= ~216).  Nothing is allocated here either: M (overwritten), tau00_out
    [batch, k, k] and info [batch] are the caller's tensors.  All calls on a device share the scratch array: do not let
    two of them overlap on the GPU.  Make the first call on a device outside any stream capture."""
    for name, t in (("M", M), ("tau00_out", tau00_out), ("info", info)):
        if t is None:
            raise LsmsError(f"lsms_tau00_onchip_static_scratch: {name} must be given (this call allocates nothing)")
    rc = lib().lsms_tau00_onchip_static_scratch(_ptr(M), n_sites, kmax, int(bool(spin_canted)), batch, _ptr(tau00_out),
                                                _ptr(info), _stream(stream))
    k = kmax * (2 if spin_canted else 1)
    if rc == LSMS_ERR_NOT_ON_CHIP:
        raise LsmsError(f"lsms_tau00_onchip_static_scratch: a {n_sites * k} x {n_sites * k} matrix does not fit the on-chip "
                        "kernel (n <= ~216); use lsms_tau00_batched with a workspace")
    if rc == LSMS_ERR_STATIC_SCRATCH_TOO_SMALL:
        raise LsmsError(f"lsms_tau00_onchip_static_scratch: batch * n = {batch * n_sites * k} exceeds the built-in scratch of "
                        f"{LSMS_STATIC_SCRATCH_WORDS} words; split the batch or use lsms_tau00_batched with a workspace")
    _check(rc, "lsms_tau00_onchip_static_scratch")
    return tau00_out, info


def lsms_solve_central_column_batched(handle: Handle, M, n_sites, kmax, spin_canted, batch, X_out=None, info=None,
                                      workspace=None, stream=None):
    """-> (X c128 [batch, k, n] with X[b, c, r] = element (row r, col c) of M^{-1} E, info)."""
    import torch
    k = kmax * (2 if spin_canted else 1)
    n = n_sites * k
    if X_out is None:
        X_out = _empty((batch, k, n), torch.complex128, M.device, stream)
    if info is None:
        info = _info(batch, M.device, stream)
    if workspace is None:
        workspace = _workspace(lsms_solve_workspace_bytes(handle, n_sites, kmax, spin_canted, batch), M.device, stream)
    _check(lib().lsms_solve_central_column_batched(handle.ptr, _ptr(M), n_sites, kmax, int(bool(spin_canted)), batch,
                                                   _ptr(X_out), _ptr(info), _ptr(workspace), workspace.numel(),
                                                   _stream(stream)), "lsms_solve_central_column_batched")
    return X_out, info


def lsms_contour_sum_batched(handle: Handle, tau00, weights, n_atoms, n_energies, k, out=None, stream=None):
    import torch
    if out is None:
        out = _empty((n_atoms, k, k), torch.complex128, tau00.device, stream)
    _check(lib().lsms_contour_sum_batched(handle.ptr, _ptr(tau00), _ptr(weights), n_atoms, n_energies, k, _ptr(out),
                                          _stream(stream)), "lsms_contour_sum_batched")
    return out


def lsms_schur_update_batched(handle: Handle, M, n, c0, kk, batch, stream=None):
    _check(lib().lsms_schur_update_batched(handle.ptr, _ptr(M), n, c0, kk, batch, _stream(stream)),
           "lsms_schur_update_batched")
    return M


class HostCall:
    """Pinned host buffers + device scratch for lsms_tau00_from_host (the end-to-end entry point)."""

    def __init__(self, handle: Handle, n_sites, lmax, spin_canted, n_species, batch, n_energies=0, device="cuda:0"):
        import torch
        self.handle = handle
        self.shape = (n_sites, lmax, bool(spin_canted), n_species, batch, n_energies)
        nspin = 2 if spin_canted else 1
        k = (lmax + 1) ** 2 * nspin
        pin = dict(pin_memory=True)
        self.delta = torch.empty((n_species, nspin, lmax + 1), dtype=torch.complex128, **pin)
        self.species = torch.empty((batch, n_sites), dtype=torch.int32, **pin)
        self.z = torch.empty((batch,), dtype=torch.complex128, **pin)
        self.site_pos = torch.empty((batch, n_sites, 3), dtype=torch.float64, **pin)
        self.moment_dir = torch.empty((batch, n_sites, 3), dtype=torch.float64, **pin)
        self.tau00 = torch.empty((batch, k, k), dtype=torch.complex128, **pin)
        self.info = torch.empty((batch,), dtype=torch.int32, **pin)
        self.scratch = _workspace(lsms_host_call_scratch_bytes(handle, n_sites, lmax, spin_canted, n_species, batch), device)
        self.h2d_bytes = 0
        self.d2h_bytes = 0

    def load(self, liz_batch) -> None:
        import torch
        self.delta.copy_(torch.from_numpy(np.ascontiguousarray(liz_batch.delta)))
        self.species.copy_(torch.from_numpy(np.ascontiguousarray(liz_batch.species)))
        self.z.copy_(torch.from_numpy(np.ascontiguousarray(liz_batch.z)))
        self.site_pos.copy_(torch.from_numpy(np.ascontiguousarray(liz_batch.site_pos)))
        self.moment_dir.copy_(torch.from_numpy(np.ascontiguousarray(liz_batch.moment_dir)))

    def run(self, stream=None):
        n_sites, lmax, canted, n_species, batch, n_energies = self.shape
        h2d, d2h = ctypes.c_size_t(0), ctypes.c_size_t(0)
        _check(lib().lsms_tau00_from_host(self.handle.ptr, _ptr(self.delta), _ptr(self.species), _ptr(self.z),
                                          _ptr(self.site_pos), _ptr(self.moment_dir) if canted else 0, lmax, n_sites,
                                          int(canted), n_species, batch, n_energies, _ptr(self.tau00), _ptr(self.info),
                                          _ptr(self.scratch), self.scratch.numel(), _stream(stream), ctypes.byref(h2d),
                                          ctypes.byref(d2h)), "lsms_tau00_from_host")
        self.h2d_bytes, self.d2h_bytes = int(h2d.value), int(d2h.value)
        return self.tau00, self.info


def device_inputs(liz_batch, device="cuda:0"):
    """Copy a synth_liz.LizBatch to device tensors (delta, species, z, site_pos, moment_dir)."""
    import torch
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(device)
    return t(liz_batch.delta), t(liz_batch.species), t(liz_batch.z), t(liz_batch.site_pos), t(liz_batch.moment_dir)


def tau00_from_liz_batch(handle: Handle, liz_batch, device="cuda:0", keep_M=False):
    """Convenience: device-resident whole path for a synth_liz.LizBatch.
    Returns (tau00 [batch,k,k] numpy indexed [b,row,col], info numpy, M copy or None)."""
    import torch
    cfg = liz_batch.cfg
    B = liz_batch.batch
    delta, species, z, pos, mom = device_inputs(liz_batch, device)
    tinv, kappa, info0 = lsms_tinv_from_phase_shifts(handle, delta, species, z, cfg.lmax, cfg.n_sites, cfg.spin_canted,
                                                     liz_batch.delta.shape[0], B)
    M, info1 = lsms_build_M_batched(handle, tinv, pos, mom if cfg.spin_canted else None, kappa, cfg.lmax, cfg.n_sites,
                                    cfg.spin_canted, B)
    Mcopy = M.clone() if keep_M else None
    tau, info = lsms_tau00_batched(handle, M, cfg.n_sites, cfg.kmax, cfg.spin_canted, B)
    torch.cuda.synchronize()
    codes = np.stack([info0.cpu().numpy(), info1.cpu().numpy(), info.cpu().numpy()])
    first = np.where(codes[0] != 0, codes[0], np.where(codes[1] != 0, codes[1], codes[2]))
    return tau.cpu().numpy().transpose(0, 2, 1).copy(), first, Mcopy
