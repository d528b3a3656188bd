"""Seeded synthetic input generators for the five BASELINE.json configs.

This module serves BOTH the CPU oracle (tests) and the CUDA path (tests, bench).
It holds none of the method's arithmetic: it only draws particle positions and
charges (numpy PCG64, fixed seeds) and names the plan parameters of each config.

The paper's own benchmark inputs (PACKMOL + periodic relaxation, stored under
msmjax/data/) are not available; these generators take the paper's
*shapes* -- random particles in a box with a minimum-distance rule 0.6*dbar,
charges summing to zero, N from 3e3 to 1e6 -- and
the concrete numbers of BASELINE.json:configs, and stand in for them.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

__all__ = ["Workload", "make_workload", "WORKLOAD_NAMES", "water_box", "rock_salt",
           "open_random", "slab_random"]


@dataclasses.dataclass
class Workload:
    """One seeded input set plus the plan parameters it is evaluated with."""
    name: str
    positions: np.ndarray          # (N, 3) float64
    charges: np.ndarray            # (N,)   float64
    box: tuple                     # (Lx, Ly, Lz)
    periodic: tuple                # (0/1, 0/1, 0/1)
    h: float                       # target finest grid spacing
    a: float                       # level-zero cutoff
    p: int                         # B-spline order
    levels: int                    # see DESIGN.md reading G4
    precision: str = "fp64"        # "fp64" | "fp32"
    note: str = ""

    @property
    def n(self) -> int:
        return int(self.positions.shape[0])

    def as_precision(self, precision: str) -> "Workload":
        """Same inputs; for fp32 the positions/charges are rounded to fp32-representable values
        (so that oracle and CUDA path start from identical numbers)."""
        if precision == "fp32":
            pos = self.positions.astype(np.float32).astype(np.float64)
            q = self.charges.astype(np.float32).astype(np.float64)
        else:
            pos, q = self.positions, self.charges
        return dataclasses.replace(self, positions=pos, charges=q, precision=precision)


# ----------------------------------------------------------------------------- generators

def open_random(n: int, edge: float, seed: int):
    """Config 1 recipe: uniform-random positions in an open cube, charges +1/-1 alternating."""
    rng = np.random.default_rng(seed)
    pos = rng.random((n, 3)) * edge
    q = np.where(np.arange(n) % 2 == 0, 1.0, -1.0)
    return pos, q


def rock_salt(ncell: int, a_lat: float, shift=None):
    """Config 2 recipe: ncell^3 conventional cubic cells of rock salt. Cations (+1) on the fcc
    sites, anions (-1) on the fcc sites shifted by (1/2, 0, 0) a_lat."""
    fcc = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.0], [0.5, 0.0, 0.5], [0.0, 0.5, 0.5]])
    cells = np.stack(np.meshgrid(np.arange(ncell), np.arange(ncell), np.arange(ncell),
                                 indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float64)
    cat = (cells[:, None, :] + fcc[None, :, :]).reshape(-1, 3)
    ani = cat + np.array([0.5, 0.0, 0.0])
    pos = np.concatenate([cat, ani], axis=0) * a_lat
    q = np.concatenate([np.ones(len(cat)), -np.ones(len(ani))])
    edge = ncell * a_lat
    if shift is not None:
        pos = pos + np.asarray(shift, dtype=np.float64)[None, :]
    pos = pos - edge * np.floor(pos / edge)
    # interleave so neighbouring indices alternate in sign (no effect on results)
    return pos, q


_Q_O, _Q_H = -0.8476, 0.4238
_R_OH = 1.0
_ANGLE_HOH = math.radians(109.47)
_VOL_PER_MOLECULE = 29.915          # A^3 at 1.0 g/cm^3 (18.015 g/mol)


def _random_rotations(rng, n):
    """Uniform random rotations from normalised 4-vectors of normals (unit quaternions)."""
    qv = rng.standard_normal((n, 4))
    qv /= np.linalg.norm(qv, axis=1, keepdims=True)
    w, x, y, z = qv.T
    rot = np.empty((n, 3, 3))
    rot[:, 0, 0] = 1 - 2 * (y * y + z * z); rot[:, 0, 1] = 2 * (x * y - z * w); rot[:, 0, 2] = 2 * (x * z + y * w)
    rot[:, 1, 0] = 2 * (x * y + z * w); rot[:, 1, 1] = 1 - 2 * (x * x + z * z); rot[:, 1, 2] = 2 * (y * z - x * w)
    rot[:, 2, 0] = 2 * (x * z - y * w); rot[:, 2, 1] = 2 * (y * z + x * w); rot[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return rot


def water_box(n_molecules: int, seed: int):
    """Configs 3/4 recipe: rigid three-site molecules (O -0.8476, 2 H +0.4238 at 1.0 A, HOH
    109.47 deg) at uniform-random positions and orientations in a periodic cubic box at
    1.0 g/cm^3, inserted sequentially (in batches) and rejected when any inter-molecular site
    pair is closer than 0.6*(V/N_sites)^(1/3) (the paper's minimum-distance rule).
    Returns (positions (3*n_molecules, 3) ordered O,H,H per molecule, charges, edge)."""
    from scipy.spatial import cKDTree  # neighbour search for the rejection test only

    n_sites = 3 * n_molecules
    edge = (n_molecules * _VOL_PER_MOLECULE) ** (1.0 / 3.0)
    dmin = 0.6 * (edge ** 3 / n_sites) ** (1.0 / 3.0)
    half = 0.5 * _ANGLE_HOH
    local = np.array([[0.0, 0.0, 0.0],
                      [_R_OH * math.sin(half), 0.0, _R_OH * math.cos(half)],
                      [-_R_OH * math.sin(half), 0.0, _R_OH * math.cos(half)]])
    rng = np.random.default_rng(seed)
    acc = np.empty((0, 3, 3))
    while acc.shape[0] < n_molecules:
        need = n_molecules - acc.shape[0]
        nb = max(64, int(1.5 * need))
        centre = rng.random((nb, 3)) * edge
        rot = _random_rotations(rng, nb)
        sites = centre[:, None, :] + np.einsum("nij,sj->nsi", rot, local)
        sites -= edge * np.floor(sites / edge)
        sites[sites >= edge] = 0.0
        flat = sites.reshape(-1, 3)
        ok = np.ones(nb, dtype=bool)
        tree_c = cKDTree(flat, boxsize=edge)
        if acc.shape[0] > 0:
            tree_a = cKDTree(acc.reshape(-1, 3), boxsize=edge)
            cnt = tree_a.query_ball_point(flat, dmin, return_length=True)
            ok &= (cnt.reshape(nb, 3).sum(axis=1) == 0)
        pairs = tree_c.query_pairs(dmin, output_type="ndarray")
        if len(pairs):
            mi, mj = pairs[:, 0] // 3, pairs[:, 1] // 3
            inter = mi != mj
            # the later-drawn molecule of every conflicting candidate pair is rejected
            ok[np.maximum(mi[inter], mj[inter])] = False
        acc = np.concatenate([acc, sites[ok][:need]], axis=0)
    pos = acc.reshape(-1, 3)
    q = np.tile(np.array([_Q_O, _Q_H, _Q_H]), n_molecules)
    return pos, q, edge


def slab_random(n: int, lx: float, ly: float, zmax: float, seed: int):
    """Config 5 recipe: x,y ~ U[0,L), z ~ U[0,zmax], q ~ U(-1,1) shifted to zero net charge."""
    rng = np.random.default_rng(seed)
    pos = np.empty((n, 3))
    pos[:, 0] = rng.random(n) * lx
    pos[:, 1] = rng.random(n) * ly
    pos[:, 2] = rng.random(n) * zmax
    q = rng.uniform(-1.0, 1.0, n)
    q -= q.mean()
    return pos, q


# ----------------------------------------------------------------------------- named configs

def _water_levels(edge: float, h: float) -> int:
    """levels so that the top grid kept as a separate stage is <= 8^3 (configs 3/4)."""
    m1 = 2 ** int(round(math.log2(edge / h)))
    return max(1, int(math.log2(m1)) - 3 + 1) if m1 > 8 else 1


def _water(name, n_molecules, seed, precision):
    pos, q, edge = water_box(n_molecules, seed)
    return Workload(name, pos, q, (edge,) * 3, (1, 1, 1), h=2.0, a=9.0, p=4,
                    levels=_water_levels(edge, 2.0), precision=precision,
                    note="water-like periodic box, 1.0 g/cm^3")


def _water_supercell(name, n_molecules_base, seed, reps, precision):
    """A reps^3 supercell of a water box plus a small random rigid displacement of every molecule
    (the way the paper builds its large systems): same density and plan parameters."""
    pos, q, edge = water_box(n_molecules_base, seed)
    rng = np.random.default_rng(seed + 1000)
    shifts = np.stack(np.meshgrid(*[np.arange(reps)] * 3, indexing="ij"), axis=-1).reshape(-1, 3) * edge
    big = (pos[None, :, :] + shifts[:, None, :]).reshape(-1, 3)
    disp = rng.uniform(-0.05, 0.05, (big.shape[0] // 3, 3))
    big = big + np.repeat(disp, 3, axis=0)
    E = edge * reps
    big -= E * np.floor(big / E)
    big[big >= E] = 0.0
    return Workload(name, big, np.tile(q, reps ** 3), (E,) * 3, (1, 1, 1), h=2.0, a=9.0, p=4,
                    levels=_water_levels(E, 2.0), precision=precision,
                    note="water-like periodic box, 1.0 g/cm^3, supercell")


# The commensurate scaling series of SURVEY.md 8(d) config 4: identical h = 2.09 at every N
# (box = 2^k * 33.44), so that linearity in N is not masked by the jumps of h that the power-of-two
# grid counts (reading G1) cause at the BASELINE points.
COMMENSURATE_SERIES = ["cfg4c_water3750", "cfg4c_water30k", "cfg4c_water240k", "cfg4c_water1920k"]
BASELINE_SWEEP = ["cfg4_water3k", "cfg4_water30k", "cfg4_water300k", "cfg4_water1m"]

WORKLOAD_NAMES = [
    "cfg1_open512", "cfg2_nacl4096", "cfg2_nacl4096_shifted", "cfg3_water30k_fp64",
    "cfg3_water30k_fp32", "cfg4_water3k", "cfg4_water30k", "cfg4_water300k", "cfg4_water1m",
    "cfg5_slab100k", "cfg4_water1m_fp64",
] + COMMENSURATE_SERIES


def make_workload(name: str) -> Workload:
    """Build one of the named workloads (BASELINE.json:configs)."""
    if name == "cfg1_open512":
        pos, q = open_random(512, 20.0, 12345)
        return Workload(name, pos, q, (20.0,) * 3, (0, 0, 0), h=2.0, a=6.0, p=4, levels=3)
    if name in ("cfg2_nacl4096", "cfg2_nacl4096_shifted"):
        shift = None
        if name.endswith("shifted"):
            shift = np.random.default_rng(2).random(3) * 5.64
        pos, q = rock_salt(8, 5.64, shift)
        return Workload(name, pos, q, (45.12,) * 3, (1, 1, 1), h=1.41, a=8.0, p=4, levels=4)
    if name == "cfg3_water30k_fp64":
        return _water(name, 10000, 3, "fp64")
    if name == "cfg3_water30k_fp32":
        return _water(name, 10000, 3, "fp32").as_precision("fp32")
    if name == "cfg4_water3k":
        return _water(name, 1000, 41, "fp32").as_precision("fp32")
    if name == "cfg4_water30k":
        return _water(name, 10000, 42, "fp32").as_precision("fp32")
    if name == "cfg4_water300k":
        return _water(name, 100000, 43, "fp32").as_precision("fp32")
    if name == "cfg4_water1m":
        return _water(name, 333333, 44, "fp32").as_precision("fp32")
    if name == "cfg4_water1m_fp64":
        return _water(name, 333333, 44, "fp64")
    if name == "cfg4c_water3750":
        return _water(name, 1250, 51, "fp32").as_precision("fp32")
    if name == "cfg4c_water30k":
        return _water(name, 10000, 52, "fp32").as_precision("fp32")
    if name == "cfg4c_water240k":
        return _water(name, 80000, 53, "fp32").as_precision("fp32")
    if name == "cfg4c_water1920k":
        return _water_supercell(name, 80000, 53, 2, "fp32").as_precision("fp32")
    if name == "cfg5_slab100k":
        pos, q = slab_random(100000, 100.0, 100.0, 40.0, 5)
        return Workload(name, pos, q, (100.0, 100.0, 40.0), (1, 1, 0), h=1.5, a=10.0, p=6,
                        levels=4)
    raise KeyError(name)
