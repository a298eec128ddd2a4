"""Input recipes for BASELINE.json configs[0..4].

Everything is generated in float64 from ``np.random.default_rng([966, cfg, dom, stream])``
(stream 0: V_loc, 1: atoms, 2: projector strengths D, 3: orbitals) and rounded ONCE to
float32 / complex64 (reading D21).  The oracle promotes these rounded values to
float64; the GPU library consumes them as they are.

The synthetic domains stand in for the paper's PbTiO3 workload:
the paper's atomic configurations, pseudopotentials and ground-state orbitals are not
available, and the hot path's cost and arithmetic do not depend on them.

No method arithmetic lives here (no finite differences, no propagator, no projection).
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Dict, Optional, Tuple

import numpy as np
import scipy.linalg

SEED_ROOT = 966
A_LATTICE = 7.4  # bohr, cubic perovskite cell (BASELINE.json configs[2])


@dataclass(frozen=True)
class DomainConfig:
    cfg: int                 # BASELINE.json config index (seed component)
    name: str
    ndom: int
    grid: Tuple[int, int, int]
    h: Tuple[float, float, float]      # bohr
    norb: int
    nocc: int                # first nocc orbitals have f=2, the rest f=0
    nsteps: int
    dt: float
    kind: str                # "toy" (cosine V, random atoms) | "perovskite"
    natoms: int = 0          # toy only
    ncell: int = 0           # perovskite: cells per edge
    laser: bool = True
    smooth_kcut: float = 0.0  # >0: low-pass the random orbitals (|k| <= kcut) before QR (reading D15)

    @property
    def ngrid(self) -> int:
        return self.grid[0] * self.grid[1] * self.grid[2]

    @property
    def dv(self) -> float:
        return self.h[0] * self.h[1] * self.h[2]

    @property
    def box(self) -> Tuple[float, float, float]:
        return tuple(n * s for n, s in zip(self.grid, self.h))

    @property
    def nproj(self) -> int:
        if self.kind == "toy":
            return 4 * self.natoms
        nc = self.ncell ** 3
        return nc * (9 + 9 + 3 * 4)

    @property
    def electrons_per_domain(self) -> float:
        return 2.0 * self.nocc


def _cube(n, hh):
    return (n, n, n), (hh, hh, hh)


CONFIGS: Dict[int, DomainConfig] = {
    0: DomainConfig(0, "toy16", 1, *_cube(16, 0.5), norb=8, nocc=8, nsteps=10, dt=0.02,
                    kind="toy", natoms=2, laser=False),
    1: DomainConfig(1, "laser32", 1, *_cube(32, 0.4), norb=64, nocc=64, nsteps=100, dt=0.02,
                    kind="toy", natoms=8),
    2: DomainConfig(2, "pto8", 8, *_cube(48, 2 * A_LATTICE / 48), norb=224, nocc=176, nsteps=20,
                    dt=0.02, kind="perovskite", ncell=2),
    3: DomainConfig(3, "pto64", 64, *_cube(48, 2 * A_LATTICE / 48), norb=224, nocc=176, nsteps=10,
                    dt=0.02, kind="perovskite", ncell=2),
    4: DomainConfig(4, "pto_large4", 4, *_cube(64, 3 * A_LATTICE / 64), norb=696, nocc=594,
                    nsteps=10, dt=0.02, kind="perovskite", ncell=3),
}


def get_config(cfg: int, **overrides) -> DomainConfig:
    """Config ``cfg`` of BASELINE.json, optionally with fields replaced (tests use smaller
    ``ndom``/``nsteps``/``grid`` variants of the same recipe)."""
    c = CONFIGS[cfg]
    return replace(c, **overrides) if overrides else c


# ----------------------------------------------------------------------------- helpers
def _rng(c: DomainConfig, dom: int, stream: int) -> np.random.Generator:
    return np.random.default_rng([SEED_ROOT, c.cfg, dom, stream])


def _coords(c: DomainConfig):
    ax = [np.arange(n, dtype=np.float64) * s for n, s in zip(c.grid, c.h)]
    return np.meshgrid(*ax, indexing="ij")  # each [nx, ny, nz]; flat index (ix*ny+iy)*nz+iz


def _min_image(delta, box_len):
    return delta - box_len * np.round(delta / box_len)


def _atoms(c: DomainConfig, dom: int):
    """Return (positions [na,3], species list) — stream 1."""
    rng = _rng(c, dom, 1)
    box = np.array(c.box)
    if c.kind == "toy":
        pos = rng.uniform(0.0, 1.0, size=(c.natoms, 3)) * box
        return pos, ["X"] * c.natoms
    frac = {"Pb": [(0.0, 0.0, 0.0)], "Ti": [(0.5, 0.5, 0.5)],
            "O": [(0.5, 0.5, 0.0), (0.5, 0.0, 0.5), (0.0, 0.5, 0.5)]}
    pos, spec = [], []
    for i in range(c.ncell):
        for j in range(c.ncell):
            for k in range(c.ncell):
                for sp in ("Pb", "Ti", "O"):
                    for f in frac[sp]:
                        pos.append([(i + f[0]) * A_LATTICE, (j + f[1]) * A_LATTICE, (k + f[2]) * A_LATTICE])
                        spec.append(sp)
    pos = np.array(pos) + rng.normal(0.0, 0.1, size=(len(pos), 3))
    pos = np.mod(pos, box)
    return pos, spec


_ANGULAR = {
    "s": [lambda x, y, z, r2: np.ones_like(x)],
    "p": [lambda x, y, z, r2: x, lambda x, y, z, r2: y, lambda x, y, z, r2: z],
    "d": [lambda x, y, z, r2: x * y, lambda x, y, z, r2: y * z, lambda x, y, z, r2: z * x,
          lambda x, y, z, r2: x * x - y * y, lambda x, y, z, r2: 3.0 * z * z - r2],
}
_SHELLS = {"X": "sp", "O": "sp", "Pb": "spd", "Ti": "spd"}
_DEPTH = {"Pb": 2.0, "Ti": 1.5, "O": 1.0}
SIGMA_PROJ = 1.0   # bohr
WIDTH_WELL = 1.0   # bohr


def _projectors(c: DomainConfig, pos, spec):
    """beta[ngrid, nproj] float64, each column normalised so that dv*sum(beta^2)=1 (reading D10/D11)."""
    X, Y, Z = _coords(c)
    box = c.box
    cols = []
    for R, sp in zip(pos, spec):
        dx = _min_image(X - R[0], box[0])
        dy = _min_image(Y - R[1], box[1])
        dz = _min_image(Z - R[2], box[2])
        r2 = dx * dx + dy * dy + dz * dz
        g = np.exp(-r2 / (2.0 * SIGMA_PROJ ** 2))
        for shell in _SHELLS[sp]:
            for ang in _ANGULAR[shell]:
                b = (ang(dx, dy, dz, r2) * g).reshape(-1)
                b /= np.sqrt(c.dv * np.sum(b * b))
                cols.append(b)
    return np.stack(cols, axis=1)


def _vloc(c: DomainConfig, dom: int, pos, spec):
    X, Y, Z = _coords(c)
    box = c.box
    if c.kind == "toy":
        rng = _rng(c, dom, 0)
        v = np.zeros(c.grid, dtype=np.float64)
        n = 0
        while n < 6:
            m = rng.integers(-2, 3, size=3)
            if not m.any():
                continue
            phi = rng.uniform(0.0, 2.0 * np.pi)
            v += 0.3 * np.cos(2.0 * np.pi * (m[0] * X / box[0] + m[1] * Y / box[1] + m[2] * Z / box[2]) + phi)
            n += 1
        return v
    v = np.zeros(c.grid, dtype=np.float64)
    for R, sp in zip(pos, spec):
        dx = _min_image(X - R[0], box[0])
        dy = _min_image(Y - R[1], box[1])
        dz = _min_image(Z - R[2], box[2])
        v -= _DEPTH[sp] * np.exp(-(dx * dx + dy * dy + dz * dz) / (2.0 * WIDTH_WELL ** 2))
    return v


def _orbitals(c: DomainConfig, dom: int):
    rng = _rng(c, dom, 3)
    g = rng.standard_normal((c.ngrid, c.norb)) + 1j * rng.standard_normal((c.ngrid, c.norb))
    if c.smooth_kcut > 0.0:
        gk = np.fft.fftn(g.reshape(*c.grid, c.norb), axes=(0, 1, 2))
        ks = [2.0 * np.pi * np.fft.fftfreq(n, d=s) for n, s in zip(c.grid, c.h)]
        KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
        mask = (KX * KX + KY * KY + KZ * KZ) <= c.smooth_kcut ** 2
        gk *= mask[..., None]
        g = np.fft.ifftn(gk, axes=(0, 1, 2)).reshape(c.ngrid, c.norb)
    # thin QR with positive-diagonal R, computed through the Cholesky factor of the Gram matrix
    # (same Q as Householder QR up to rounding; ~10x faster for these well-conditioned tall matrices)
    low = np.linalg.cholesky(g.conj().T @ g)
    q = scipy.linalg.solve_triangular(low, g.conj().T, lower=True, overwrite_b=True, check_finite=False).conj().T
    return q / np.sqrt(c.dv)


def laser_samples(c: DomainConfig, nsteps: Optional[int] = None, t0: float = 0.0) -> np.ndarray:
    """A[nsteps, 1, 3] float64: x-polarised sin^2 pulse sampled at the step midpoints
    t_n + dt/2 (reading D7): peak 0.1 a.u., omega 0.057 a.u., duration 100*dt."""
    n = c.nsteps if nsteps is None else nsteps
    A = np.zeros((n, 1, 3), dtype=np.float64)
    if not c.laser:
        return A
    T = 100.0 * c.dt
    t = t0 + (np.arange(n) + 0.5) * c.dt
    inside = (t >= 0.0) & (t <= T)
    A[:, 0, 0] = np.where(inside, 0.1 * np.sin(np.pi * t / T) ** 2 * np.cos(0.057 * (t - T / 2.0)), 0.0)
    return A


def generate_domain(c: DomainConfig, dom: int) -> Dict[str, np.ndarray]:
    """All arrays of one domain, rounded once to the storage precision the library takes."""
    pos, spec = _atoms(c, dom)
    beta = _projectors(c, pos, spec)
    D = _rng(c, dom, 2).uniform(-1.0, 1.0, size=beta.shape[1])
    vloc = _vloc(c, dom, pos, spec)
    psi = _orbitals(c, dom)
    occ = np.zeros(c.norb, dtype=np.float64)
    occ[: c.nocc] = 2.0
    return {
        "psi": psi.astype(np.complex64).reshape(*c.grid, c.norb),
        "occ": occ,
        "vloc": vloc.astype(np.float32),
        "beta": beta.astype(np.float32),
        "D": D,
        "atoms": pos,
    }


def generate(c: DomainConfig, workers: int = 1) -> Dict[str, np.ndarray]:
    """Stack ``generate_domain`` over all ``c.ndom`` domains and add the laser samples.
    ``workers`` > 1 builds domains in a thread pool (numpy's RNG, BLAS and LAPACK release the GIL);
    the result does not depend on it because every domain has its own seed."""
    if workers > 1 and c.ndom > 1:
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(max_workers=workers) as ex:
            doms = list(ex.map(lambda d: generate_domain(c, d), range(c.ndom)))
    else:
        doms = [generate_domain(c, d) for d in range(c.ndom)]
    out = {k: np.stack([d[k] for d in doms], axis=0) for k in ("psi", "occ", "vloc", "beta", "D")}
    out["A"] = laser_samples(c)
    return out
