"""SURVEY.md section 5 (sanitizer row), the part that needs no GPU: the CPU oracle compiled with
-fsanitize=address,undefined runs its tiny-LIZ routes clean (no out-of-bounds access, no undefined behaviour).
compute-sanitizer for the CUDA path is closed on the GPU pool, so this covers the checker only."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r"""
import numpy as np
import oracle, synth_liz as sl
assert oracle.lib()._name.endswith("liblsms_oracle_san.so")
T = oracle.gaunt_table(3)
assert np.isfinite(T).all()
batch = sl.make_batch("T").select([0, 13, 31])
cfg = batch.cfg
tau, info = oracle.tau00_batched(batch, "double")
assert not info.any()
M = oracle.assemble_M(cfg.n_sites, cfg.lmax, cfg.spin_canted, batch.site_pos[0], batch.species[0], batch.delta, batch.moment_dir[0], batch.z[0])
t_full = oracle.tau00_full(M, cfg.k, "long double")
t_schur = oracle.tau00_schur(M, cfg.k)
t_ref = oracle.tau00_refined(M, cfg.k, 2)
inv = oracle.inverse_gauss_jordan(M)
for t in (t_schur, t_ref, inv[-cfg.k:, -cfg.k:], tau[0]):
    assert np.linalg.norm(t - t_full) < 1e-11 * np.linalg.norm(t_full)
c = sl.make_batch(sl.custom_config(13, 2, True, n_energies=2))
tc, ic = oracle.tau00_batched(c, "long double")
assert not ic.any()
w = sl.contour_weights("semicircle", 3)
s = oracle.contour_sum(tau.reshape(1, 3, cfg.k, cfg.k), w)
assert np.isfinite(s).all()
print("sanitized oracle ok")
"""


def test_oracle_runs_clean_under_asan_and_ubsan(tmp_path):
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    ubsan = subprocess.run(["gcc", "-print-file-name=libubsan.so"], capture_output=True, text=True).stdout.strip()
    if not (os.path.isabs(asan) and os.path.exists(asan) and os.path.isabs(ubsan) and os.path.exists(ubsan)):
        pytest.skip("libasan / libubsan not installed")
    lib = str(tmp_path / "liblsms_oracle_san.so")
    subprocess.check_call(["g++", "-O1", "-g", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-fno-omit-frame-pointer",
                           "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                           "-o", lib, os.path.join(ROOT, "oracle", "lsms_oracle.cpp")])
    env = dict(os.environ, LSMS_ORACLE_LIB=lib, LD_PRELOAD=f"{asan}:{ubsan}", PYTHONPATH=ROOT, OMP_NUM_THREADS="2",
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:exitcode=97", UBSAN_OPTIONS="halt_on_error=1:exitcode=98:print_stacktrace=1")
    r = subprocess.run([sys.executable, "-c", SCRIPT], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, (r.returncode, r.stderr[-3000:])
    assert "sanitized oracle ok" in r.stdout
    assert "AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr, r.stderr[-3000:]
