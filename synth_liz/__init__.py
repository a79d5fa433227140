"""Seeded synthetic-LIZ input generator shared by the oracle side and the CUDA side.

This module produces INPUTS ONLY (geometry, occupancies, phase shifts, moment
directions, contour energies).  It holds none of the method's arithmetic: no
kappa = sqrt(z), no t-matrix, no structure constants, no elimination.  Both
`oracle/` and `paper_2308_16317_b200/` start from what is generated here and
each does its own arithmetic.

Recipe: SURVEY.md section 8(d) ("Synthetic inputs"), readings A5-A12, A19, A20
of section 8(c); configs are BASELINE.json `configs[0..4]` (T, M, P, C, H).
The paper's real workloads (NiAu / CoCrFeMnNi through MuST
with physical potentials) are not available; these inputs take their shapes
(FCC LIZ, N_LIZ up to 135, l_max 3-4, +/- spin canting, complex double on an
energy contour) and stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

BOHR_PER_ANGSTROM = 1.0 / 0.529177210903  # A5: lengths in Bohr
A_FCC_BOHR = 3.8 * BOHR_PER_ANGSTROM      # configs[0]: a = 3.8 Angstrom
BASE_SEED = 230816317                     # section 8(d)

_MASK = (1 << 64) - 1


class SplitMix64:
    """SplitMix64 stream; u = ((x >> 11) + 1/2) * 2^-53 in (0,1) (reading A20)."""

    def __init__(self, seed: int):
        self.s = seed & _MASK

    def next_u64(self) -> int:
        self.s = (self.s + 0x9E3779B97F4A7C15) & _MASK
        z = self.s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
        return z ^ (z >> 31)

    def uniform(self) -> float:
        return ((self.next_u64() >> 11) + 0.5) * (2.0 ** -53)

    def normal_pair(self) -> tuple[float, float]:
        """Box-Muller from two uniforms."""
        u1, u2 = self.uniform(), self.uniform()
        r = np.sqrt(-2.0 * np.log(u1))
        return float(r * np.cos(2.0 * np.pi * u2)), float(r * np.sin(2.0 * np.pi * u2))


@dataclass(frozen=True)
class LizConfig:
    name: str
    index: int          # position in BASELINE.json configs
    n_sites: int
    lmax: int
    spin_canted: bool
    n_atoms: int
    n_energies: int
    contour: str        # "semicircle" (A6) or "arc" (A7)
    ni_fraction: float = 0.5   # P(site is Ni): 1/2 for BASELINE.json's configs (A9), 0.3 for the paper's NiAu

    @property
    def kmax(self) -> int:
        return (self.lmax + 1) ** 2

    @property
    def k(self) -> int:
        return self.kmax * (2 if self.spin_canted else 1)

    @property
    def n(self) -> int:
        return self.n_sites * self.k

    @property
    def batch(self) -> int:
        return self.n_atoms * self.n_energies

    @property
    def n_spin(self) -> int:
        return 2 if self.spin_canted else 1


CONFIGS = {
    "T": LizConfig("tiny", 0, 13, 3, False, 1, 32, "semicircle"),
    "M": LizConfig("mid", 1, 55, 3, False, 16, 32, "semicircle"),
    "P": LizConfig("production", 2, 135, 3, False, 4, 32, "semicircle"),
    "C": LizConfig("spin-canted", 3, 135, 3, True, 2, 32, "semicircle"),
    "H": LizConfig("high-l", 4, 135, 4, True, 1, 24, "arc"),
    # the paper's own NiAu shapes (30 % Ni / 70 % Au, N_LIZ = 249, l_max = 4):
    # rank 6225 and, spin-canted, 12450.  Not in BASELINE.json's configs; batch sizes chosen to fit one GPU.
    "N": LizConfig("NiAu-249", 5, 249, 4, False, 1, 24, "semicircle", 0.3),
    "NC": LizConfig("NiAu-249-canted", 6, 249, 4, True, 1, 12, "semicircle", 0.3),
}

FCC_SHELL_CLOSURES = (1, 13, 19, 43, 55, 79, 87, 135, 141, 177, 201, 225, 249, 321)


def fcc_liz_lattice_points(n_sites: int) -> np.ndarray:
    """Integer FCC points (i,j,k), i+j+k even, sorted by (d^2, i, j, k) (reading A8).

    Returns int64 [n_sites,3]; row 0 is the central site (0,0,0).  n_sites must
    close a neighbour shell.
    """
    if n_sites not in FCC_SHELL_CLOSURES:
        raise ValueError(f"n_sites={n_sites} does not close an FCC shell")
    r = 1
    while True:
        g = np.arange(-r, r + 1)
        i, j, k = np.meshgrid(g, g, g, indexing="ij")
        pts = np.stack([i.ravel(), j.ravel(), k.ravel()], axis=1)
        pts = pts[(pts.sum(axis=1) % 2) == 0]
        d2 = (pts ** 2).sum(axis=1)
        # every point with d2 <= r^2 is inside the cube, so the first entries are complete
        order = np.lexsort((pts[:, 2], pts[:, 1], pts[:, 0], d2))
        pts, d2 = pts[order], d2[order]
        if len(pts) > n_sites and d2[n_sites] <= r * r and d2[n_sites - 1] <= r * r:
            assert d2[n_sites] > d2[n_sites - 1], "n_sites does not close a shell"
            return pts[:n_sites].astype(np.int64)
        r += 1


def site_positions(n_sites: int, a_bohr: float = A_FCC_BOHR) -> np.ndarray:
    """Cartesian positions in Bohr, float64 [n_sites,3]; site 0 = central."""
    return fcc_liz_lattice_points(n_sites).astype(np.float64) * (a_bohr / 2.0)


def contour_energies(kind: str, n_points: int) -> np.ndarray:
    """Complex energies z_q in Ry on the circle centre 0.1, radius 0.6 (A6 / A7).

    semicircle: theta_q = pi (1 - x_q)/2,   x_q Gauss-Legendre nodes ascending.
    arc:        theta_q = (pi/4)(1 - x_q)/2.
    The GL nodes are input geometry (a library routine), not method arithmetic.
    """
    x, _ = np.polynomial.legendre.leggauss(n_points)
    x = np.sort(x)
    if kind == "semicircle":
        theta = np.pi * (1.0 - x) / 2.0
    elif kind == "arc":
        theta = (np.pi / 4.0) * (1.0 - x) / 2.0
    else:
        raise ValueError(kind)
    return 0.1 + 0.6 * np.exp(1j * theta)


def contour_weights(kind: str, n_points: int) -> np.ndarray:
    """Complex quadrature weights w_q with  int_{-0.5}^{0.7} f(z) dz ~= sum_q w_q f(z_q)  along the contour of
    `contour_energies` (same node order): z = 0.1 + 0.6 e^{i theta}, theta = theta_max (1 - x)/2, so
    w_q = omega_q * dz/dx = -i * 0.6 e^{i theta_q} * (theta_max / 2) * omega_q  with omega_q the Gauss-Legendre
    weights.  Like the nodes, the rule is input data for the reduction of SURVEY 8(f) f4, not method arithmetic."""
    x, om = np.polynomial.legendre.leggauss(n_points)
    order = np.argsort(x)
    x, om = x[order], om[order]
    tmax = {"semicircle": np.pi, "arc": np.pi / 4.0}[kind]
    theta = tmax * (1.0 - x) / 2.0
    return (-1j * 0.6 * np.exp(1j * theta) * (tmax / 2.0) * om).astype(np.complex128)


def phase_shift_table(cfg: LizConfig) -> np.ndarray:
    """delta[species(0=Ni,1=Au)][spin][l], complex128 (A10, A11).

    Re ~ U(0,1.5), Im ~ U(0,0.05); one draw per (config, species, spin, l) from
    stream 0.  Config H: Au d-channel Re delta_2 = 1.4 for both spins (Im drawn).
    """
    rng = SplitMix64(BASE_SEED + 1000 * cfg.index + 0)
    d = np.zeros((2, cfg.n_spin, cfg.lmax + 1), dtype=np.complex128)
    for sp in range(2):
        for s in range(cfg.n_spin):
            for l in range(cfg.lmax + 1):
                re = 1.5 * rng.uniform()
                im = 0.05 * rng.uniform()
                d[sp, s, l] = complex(re, im)
    if cfg.name == "high-l":
        d[1, :, 2] = 1.4 + 1j * d[1, :, 2].imag
    return d


def atom_occupancy_and_moments(cfg: LizConfig, atom: int) -> tuple[np.ndarray, np.ndarray]:
    """Per central atom: species int32 [n_sites], Ni with probability cfg.ni_fraction (1/2: A9) and unit
    moment directions float64 [n_sites,3] (A12, isotropic).  Stream 1+atom."""
    rng = SplitMix64(BASE_SEED + 1000 * cfg.index + 1 + atom)
    species = np.zeros(cfg.n_sites, dtype=np.int32)
    for i in range(cfg.n_sites):
        species[i] = 1 if rng.uniform() >= cfg.ni_fraction else 0
    mom = np.zeros((cfg.n_sites, 3), dtype=np.float64)
    for i in range(cfg.n_sites):
        a, b = rng.normal_pair()
        c, _ = rng.normal_pair()
        v = np.array([a, b, c])
        mom[i] = v / np.linalg.norm(v)
    return species, mom


@dataclass
class LizBatch:
    cfg: LizConfig
    site_pos: np.ndarray     # float64 [batch, n_sites, 3] Bohr, site 0 central
    species: np.ndarray      # int32   [batch, n_sites]
    moment_dir: np.ndarray   # float64 [batch, n_sites, 3] (unit; used iff spin_canted)
    delta: np.ndarray        # complex128 [2, n_spin, lmax+1]
    z: np.ndarray            # complex128 [batch] energies, batch index = atom*n_E + e (A19)

    def select(self, items) -> "LizBatch":
        items = np.asarray(items, dtype=np.int64)
        return LizBatch(self.cfg, np.ascontiguousarray(self.site_pos[items]),
                        np.ascontiguousarray(self.species[items]),
                        np.ascontiguousarray(self.moment_dir[items]),
                        self.delta, np.ascontiguousarray(self.z[items]))

    @property
    def batch(self) -> int:
        return int(self.z.shape[0])


def make_batch(cfg: LizConfig | str, n_atoms: int | None = None,
               n_energies: int | None = None, atom_offset: int = 0) -> LizBatch:
    """Full synthetic batch of a config (optionally fewer atoms / energies; atom_offset shifts the
    central-atom index, i.e. the occupancy/moment streams -- used to give every rank its own atoms)."""
    if isinstance(cfg, str):
        cfg = CONFIGS[cfg]
    na = cfg.n_atoms if n_atoms is None else n_atoms
    zq = contour_energies(cfg.contour, cfg.n_energies)
    if n_energies is not None:
        zq = zq[:n_energies]
    ne = len(zq)
    pos = site_positions(cfg.n_sites)
    delta = phase_shift_table(cfg)
    B = na * ne
    site_pos = np.broadcast_to(pos, (B, cfg.n_sites, 3)).copy()
    species = np.zeros((B, cfg.n_sites), dtype=np.int32)
    mom = np.zeros((B, cfg.n_sites, 3), dtype=np.float64)
    z = np.zeros(B, dtype=np.complex128)
    for a in range(na):
        sp, m = atom_occupancy_and_moments(cfg, a + atom_offset)
        species[a * ne:(a + 1) * ne] = sp
        mom[a * ne:(a + 1) * ne] = m
        z[a * ne:(a + 1) * ne] = zq
    return LizBatch(cfg, site_pos, species, mom, delta, z)


def custom_config(n_sites: int, lmax: int, spin_canted: bool, n_atoms: int = 1,
                  n_energies: int = 4, contour: str = "semicircle", index: int = 9,
                  name: str = "custom") -> LizConfig:
    """A reduced-size config for tests (same recipe, different shape)."""
    return LizConfig(name, index, n_sites, lmax, spin_canted, n_atoms, n_energies, contour)


def random_dense_matrices(batch: int, n: int, seed: int) -> np.ndarray:
    """Random well-conditioned non-LIZ matrices, complex128 [batch, n, n] C-order
    holding COLUMN-MAJOR data (element (r,c) of item b at [b, c, r]).  Used to
    drive `lsms_tau00_batched` directly (last bullet)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    a = rng.standard_normal((batch, n, n)) + 1j * rng.standard_normal((batch, n, n))
    a += 0.5 * np.sqrt(n) * np.eye(n)[None] * np.exp(1j * rng.uniform(0, 2 * np.pi, (batch, 1, 1)))
    return np.ascontiguousarray(a.astype(np.complex128))
