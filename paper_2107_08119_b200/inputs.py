"""Seeded synthetic inputs for the NEP hot path (BASELINE.json configs C0..C4).

This module is the ONLY code shared by the oracle tests and the CUDA path.  It
holds none of the method's arithmetic (no radial functions, no descriptor, no
network): just lattices, jitter, Maxwell-Boltzmann velocities and uniform
weights, all drawn from a self-contained counter-based SplitMix64 stream so the
arrays do not depend on the numpy version.

The paper's own speed test used 8000-atom Si / PbTe cells with *trained*
potentials; neither the weights nor the DFT datasets exist here,
so these seeded stand-ins take the paper's shapes (crystalline Si, a-Si at Si
density, rock-salt PbTe; 64 ... 2M atoms) and
Table-I-like hyper-parameters.  Recipe: DESIGN.md section 4.

Conventions
-----------
* positions / velocities: float64 array of shape (3, N), SoA  x[N] | y[N] | z[N]
* units: Angstrom, fs, amu, eV, K
* parameter blob order (reading Q7):
      w1[H][D] row-major | b1[H] | w2[H] | b2        (N_par = (D+2)H+1, Eq. 26)
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

# physical constants used only for the velocity draw / unit conversion
KB_EV_PER_K = 8.617333262e-5          # CODATA 2018
AMU_A2_FS2_IN_EV = 103.642697         # 1 amu*A^2/fs^2 in eV

MASS = {"Si": 28.0855, "Pb": 207.2, "Te": 127.60}
ZNUM = {"Si": 14, "Pb": 82, "Te": 52}

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64(seed: int, n: int, offset: int = 0) -> np.ndarray:
    """Outputs offset .. offset+n-1 of the SplitMix64 stream started at `seed`."""
    with np.errstate(over="ignore"):
        k = np.arange(offset + 1, offset + n + 1, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + k * _GAMMA
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, n: int, offset: int = 0) -> np.ndarray:
    """n doubles in [0, 1): (x >> 11) * 2^-53."""
    return (splitmix64(seed, n, offset) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal(seed: int, n: int, offset: int = 0) -> np.ndarray:
    """n standard normals: Box-Muller on consecutive uniform pairs (u1,u2) ->
    (sqrt(-2 ln(1-u1)) cos 2 pi u2, sqrt(-2 ln(1-u1)) sin 2 pi u2)."""
    m = (n + 1) // 2
    u = uniform01(seed, 2 * m, 2 * offset)
    rad = np.sqrt(-2.0 * np.log1p(-u[0::2]))
    ang = 2.0 * math.pi * u[1::2]
    out = np.empty(2 * m)
    out[0::2] = rad * np.cos(ang)
    out[1::2] = rad * np.sin(ang)
    return out[:n]


# --------------------------------------------------------------------------- lattices
_DIAMOND_BASIS = np.array(
    [[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0],
     [.25, .25, .25], [.25, .75, .75], [.75, .25, .75], [.75, .75, .25]])
_FCC = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]])


def _lattice(basis: np.ndarray, a: float, cells) -> np.ndarray:
    """cell x slowest, then y, z, then basis; returns (N,3)."""
    nx, ny, nz = cells
    ix, iy, iz = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    origin = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1).astype(np.float64)
    r = (origin[:, None, :] + basis[None, :, :]).reshape(-1, 3) * a
    return r


def _jitter_wrap(r: np.ndarray, sigma: float, seed: int, box: np.ndarray) -> np.ndarray:
    """atom-major N x 3 normals * sigma, then wrap into [0, L)."""
    n = r.shape[0]
    r = r + sigma * normal(seed, 3 * n).reshape(n, 3)
    r = r - box * np.floor(r / box)
    r = np.where(r >= box, r - box, r)      # guard the floor() rounding corner
    return r


def maxwell_boltzmann(mass: np.ndarray, temperature: float, seed: int) -> np.ndarray:
    """(3,N) velocities in A/fs: N(0, kT/m) per component -> remove centre-of-mass
    velocity -> rescale to exactly `temperature` with 3N-3 degrees of freedom."""
    n = mass.shape[0]
    z = normal(seed, 3 * n).reshape(n, 3)
    v = z * np.sqrt(KB_EV_PER_K * temperature / (mass * AMU_A2_FS2_IN_EV))[:, None]
    v -= (mass[:, None] * v).sum(0) / mass.sum()
    ke = 0.5 * AMU_A2_FS2_IN_EV * (mass[:, None] * v * v).sum()
    t_now = 2.0 * ke / ((3 * n - 3) * KB_EV_PER_K)
    v *= math.sqrt(temperature / t_now)
    return np.ascontiguousarray(v.T)


def amorphous(n: int, side: float, dmin: float, seed: int) -> np.ndarray:
    """Random sequential insertion: uniform point, accept iff every accepted atom
    is >= dmin away (minimum image).  Returns (n,3).  A cell grid only speeds up
    the rejection test; the accepted sequence depends on the stream alone."""
    ncell = max(1, int(side / dmin))
    edge = side / ncell
    grid: dict[tuple[int, int, int], list[int]] = {}
    pts = np.empty((n, 3))
    count = 0
    drawn = 0
    chunk = 4096
    while count < n:
        u = uniform01(seed, 3 * chunk, 3 * drawn).reshape(chunk, 3) * side
        drawn += chunk
        for p in u:
            c = tuple(int(v) for v in np.minimum((p / edge).astype(np.int64), ncell - 1))
            ok = True
            for dx in (-1, 0, 1):
                for dy in (-1, 0, 1):
                    for dz in (-1, 0, 1):
                        key = ((c[0] + dx) % ncell, (c[1] + dy) % ncell, (c[2] + dz) % ncell)
                        for j in grid.get(key, ()):
                            d = pts[j] - p
                            d -= side * np.rint(d / side)
                            if d @ d < dmin * dmin:
                                ok = False
                                break
                        if not ok:
                            break
                    if not ok:
                        break
                if not ok:
                    break
            if ok:
                pts[count] = p
                grid.setdefault(c, []).append(count)
                count += 1
                if count == n:
                    break
    return pts


# --------------------------------------------------------------------------- weights
def descriptor_dim(n_max_r: int, n_max_a: int, l_max: int) -> int:
    return (n_max_r + 1) + (n_max_a + 1) * l_max


def make_params(dim: int, n_neurons: int, seed: int) -> np.ndarray:
    """U(-1,1)/sqrt(fan_in); fan_in = D for w1 and b1, H for w2 and b2."""
    n_par = (dim + 2) * n_neurons + 1
    u = 2.0 * uniform01(seed, n_par) - 1.0
    scale = np.empty(n_par)
    n1 = dim * n_neurons + n_neurons
    scale[:n1] = 1.0 / math.sqrt(dim)
    scale[n1:] = 1.0 / math.sqrt(n_neurons)
    return u * scale


# --------------------------------------------------------------------------- configs
@dataclasses.dataclass
class Workload:
    name: str
    pos: np.ndarray          # (3,N) float64
    vel: np.ndarray          # (3,N) float64
    types: np.ndarray        # (N,) int32
    box: np.ndarray          # (3,) float64
    rc_r: float
    rc_a: float
    n_max_r: int             # paper convention: n = 0..n_max inclusive (Eq. 16)
    n_max_a: int
    l_max: int
    n_neurons: int
    atomic_numbers: np.ndarray   # (n_types,) int32
    masses: np.ndarray           # (n_types,) float64
    params: np.ndarray           # (N_par,) float64
    dt: float = 1.0
    n_steps: int = 0

    @property
    def n_atoms(self) -> int:
        return self.pos.shape[1]

    @property
    def dim(self) -> int:
        return descriptor_dim(self.n_max_r, self.n_max_a, self.l_max)


def _si_workload(name, cells, sigma, seed_pos, seed_vel, n_max=7, n_steps=0, weights_seed=1):
    a = 5.431
    box = np.array(cells, dtype=np.float64) * a
    r = _jitter_wrap(_lattice(_DIAMOND_BASIS, a, cells), sigma, seed_pos, box)
    n = r.shape[0]
    types = np.zeros(n, dtype=np.int32)
    masses = np.array([MASS["Si"]])
    vel = maxwell_boltzmann(masses[types], 300.0, seed_vel)
    dim = descriptor_dim(n_max, n_max, 4)
    return Workload(name, np.ascontiguousarray(r.T), vel, types, box, 5.0, 4.0, n_max, n_max, 4, 30,
                    np.array([ZNUM["Si"]], dtype=np.int32), masses, make_params(dim, 30, weights_seed),
                    1.0, n_steps)


def config0(n_max: int = 7) -> Workload:
    """C0 tiny Si, 64 atoms; n_max=7 -> D=40 (primary reading Q1), n_max=8 -> D=45."""
    return _si_workload("C0_si64", (2, 2, 2), 0.05, 0, 3, n_max)


def config1(n_max: int = 7) -> Workload:
    return _si_workload("C1_si4096", (8, 8, 8), 0.1, 2, 3, n_max, n_steps=100)


def config2(n_max: int = 7, n_atoms: int = 8000, side: float = 54.3) -> Workload:
    box = np.array([side] * 3)
    r = amorphous(n_atoms, side, 2.0, 4)
    types = np.zeros(n_atoms, dtype=np.int32)
    masses = np.array([MASS["Si"]])
    vel = maxwell_boltzmann(masses[types], 300.0, 3)
    dim = descriptor_dim(n_max, n_max, 4)
    return Workload("C2_aSi%d" % n_atoms, np.ascontiguousarray(r.T), vel, types, box, 5.0, 4.0, n_max, n_max, 4, 30,
                    np.array([ZNUM["Si"]], dtype=np.int32), masses, make_params(dim, 30, 1), 1.0, 100)


def config3(cells=(20, 20, 20), n_max: int = 7) -> Workload:
    """C3 rock-salt PbTe: Pb (type 0) on fcc, Te (type 1) on fcc+(1/2,0,0); Eq. 19 weighting."""
    a = 6.46
    box = np.array(cells, dtype=np.float64) * a
    basis = np.concatenate([_FCC, _FCC + np.array([.5, 0, 0])])
    r = _jitter_wrap(_lattice(basis, a, cells), 0.1, 5, box)
    n = r.shape[0]
    types = np.tile(np.array([0, 0, 0, 0, 1, 1, 1, 1], dtype=np.int32), n // 8)
    masses = np.array([MASS["Pb"], MASS["Te"]])
    vel = maxwell_boltzmann(masses[types], 300.0, 6)
    dim = descriptor_dim(n_max, n_max, 4)
    return Workload("C3_pbte%d" % n, np.ascontiguousarray(r.T), vel, types, box, 6.0, 4.5, n_max, n_max, 4, 30,
                    np.array([ZNUM["Pb"], ZNUM["Te"]], dtype=np.int32), masses, make_params(dim, 30, 7),
                    1.0, 1000)


C4_CELLS = {32768: (16, 16, 16), 262144: (32, 32, 32), 884736: (48, 48, 48),
            1048576: (64, 64, 32), 2097152: (64, 64, 64)}


def config4(n_atoms: int = 1048576, n_max: int = 7) -> Workload:
    """C4 large Si sweep.  1048576 atoms = 64x64x32 conventional cells (reading Q17)."""
    cells = C4_CELLS[n_atoms]
    w = _si_workload("C4_si%d" % n_atoms, cells, 0.1, 8, 9, n_max, n_steps=1000)
    return w


def si_cells(cells, sigma=0.1, seed_pos=8, seed_vel=9, n_max=7) -> Workload:
    """Any diamond-Si replica with the C4 seeds (used for bounded oracle samples)."""
    return _si_workload("si_%dx%dx%d" % tuple(cells), tuple(cells), sigma, seed_pos, seed_vel, n_max)


# --------------------------------------------------------------------------- Table I shapes
def _silicene_sheet(nx: int, ny: int, a: float = 3.87, buckling: float = 0.45, vacuum: float = 20.0):
    """Buckled honeycomb sheet in an orthorhombic box: rectangular cell (a, a sqrt 3) with 4 atoms, the two
    sublattices displaced by +-buckling/2 along z, a vacuum layer above (the 2-D geometry of PAPER.md:322)."""
    b = a * math.sqrt(3.0)
    basis = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.0], [0.0, 1.0 / 3.0, 1.0], [0.5, 5.0 / 6.0, 1.0]])
    ix, iy = np.meshgrid(np.arange(nx), np.arange(ny), indexing="ij")
    origin = np.stack([ix.ravel(), iy.ravel()], axis=1).astype(np.float64)
    xy = (origin[:, None, :] + basis[None, :, :2]).reshape(-1, 2) * np.array([a, b])
    z = 0.5 * vacuum + buckling * (np.tile(basis[:, 2], nx * ny) - 0.5)
    r = np.concatenate([xy, z[:, None]], axis=1)
    return r, np.array([nx * a, ny * b, vacuum])


def table1(which: str, cells=None, sigma: float = 0.1) -> Workload:
    """The paper's three model SHAPES (Table I; N_des/N_par at PAPER.md:361) with seeded
    random weights (the trained ones do not exist here), on cells of the size the paper timed (8000-atom bulk
    Si and PbTe, 6000-atom silicene):
      "si"        n_max 15/15, r_c 5/5 A,     l_max 4, N_neu 50  -> 80-50-1   diamond Si, 10^3 cells
      "silicene"  n_max 12/12, r_c 5.5/5.5 A, l_max 4, N_neu 40  -> 65-40-1   buckled 2-D sheet + vacuum, 30 x 50 cells
      "pbte"      n_max 12/6,  r_c 8/4 A,     l_max 4, N_neu 40  -> 41-40-1   rock-salt PbTe, 10^3 cells, Eq. 19"""
    if which == "si":
        cells = cells or (10, 10, 10)
        a = 5.431
        box = np.array(cells, dtype=np.float64) * a
        r = _jitter_wrap(_lattice(_DIAMOND_BASIS, a, cells), sigma, 21, box)
        types = np.zeros(r.shape[0], dtype=np.int32)
        masses, zs = np.array([MASS["Si"]]), np.array([ZNUM["Si"]], dtype=np.int32)
        hyp = (5.0, 5.0, 15, 15, 4, 50)
    elif which == "silicene":
        cells = cells or (30, 50)
        r0, box = _silicene_sheet(cells[0], cells[1])
        r = _jitter_wrap(r0, sigma, 22, box)
        types = np.zeros(r.shape[0], dtype=np.int32)
        masses, zs = np.array([MASS["Si"]]), np.array([ZNUM["Si"]], dtype=np.int32)
        hyp = (5.5, 5.5, 12, 12, 4, 40)
    elif which == "pbte":
        cells = cells or (10, 10, 10)
        a = 6.46
        box = np.array(cells, dtype=np.float64) * a
        basis = np.concatenate([_FCC, _FCC + np.array([.5, 0, 0])])
        r = _jitter_wrap(_lattice(basis, a, cells), sigma, 23, box)
        types = np.tile(np.array([0, 0, 0, 0, 1, 1, 1, 1], dtype=np.int32), r.shape[0] // 8)
        masses, zs = np.array([MASS["Pb"], MASS["Te"]]), np.array([ZNUM["Pb"], ZNUM["Te"]], dtype=np.int32)
        hyp = (8.0, 4.0, 12, 6, 4, 40)
    else:
        raise ValueError(which)
    vel = maxwell_boltzmann(masses[types], 300.0, 24)
    dim = descriptor_dim(hyp[2], hyp[3], hyp[4])
    return Workload("table1_" + which, np.ascontiguousarray(r.T), vel, types, box, hyp[0], hyp[1], hyp[2], hyp[3],
                    hyp[4], hyp[5], zs, masses, make_params(dim, hyp[5], 25), 1.0, 100)


# --------------------------------------------------------------------------- training-side inputs
@dataclasses.dataclass
class TrainingSet:
    """Small periodic structures concatenated into one system: atoms first[n] .. first[n+1]-1 belong
    to structure n, which has its own orthorhombic box boxes[n]."""
    first: np.ndarray        # (S+1,) int64
    pos: np.ndarray          # (3, N) float64, concatenated
    types: np.ndarray        # (N,) int32
    boxes: np.ndarray        # (S, 3) float64

    @property
    def n_structures(self) -> int:
        return self.boxes.shape[0]

    @property
    def n_atoms(self) -> int:
        return self.pos.shape[1]


def training_set(n_structures: int = 24, seed: int = 50, cells=(2, 2, 2), material: str = "si") -> TrainingSet:
    """Seeded stand-in for a training set of ~100-atom structures: diamond-Si supercells with a
    per-structure lattice constant in [5.35, 5.60] A (strain), an anisotropic stretch of up to 2 % per axis and a Gaussian
    jitter of 0.03-0.15 A, every third structure with a vacancy (63 atoms).  Every box edge exceeds 2 r_c^R = 10 A."""
    u = uniform01(seed, 8 * n_structures)
    pos, boxes, first, types = [], [], [0], []
    pbte = material == "pbte"      # rock-salt PbTe, a in [6.35, 6.60] A (every edge > 2 x 6.0 A), Pb = type 0, Te = type 1
    basis = np.concatenate([_FCC, _FCC + np.array([.5, 0, 0])]) if pbte else _DIAMOND_BASIS
    for n in range(n_structures):
        a = (6.35 if pbte else 5.35) + 0.25 * u[8 * n]
        stretch = 1.0 + 0.02 * (2.0 * u[8 * n + 1:8 * n + 4] - 1.0)
        sigma = 0.03 + 0.12 * u[8 * n + 4]
        box = np.array(cells, dtype=np.float64) * a * stretch
        r = _lattice(basis, a, cells) * stretch
        ty = np.tile(np.array([0, 0, 0, 0, 1, 1, 1, 1], dtype=np.int32), r.shape[0] // 8) if pbte else np.zeros(r.shape[0], dtype=np.int32)
        if n % 3 == 2:
            k = int(u[8 * n + 5] * r.shape[0])
            r = np.delete(r, k, axis=0); ty = np.delete(ty, k)
        r = _jitter_wrap(r, sigma, seed + 1000 + n, box)
        pos.append(r); boxes.append(box); first.append(first[-1] + r.shape[0]); types.append(ty)
    allpos = np.concatenate(pos, axis=0)
    return TrainingSet(np.array(first, dtype=np.int64), np.ascontiguousarray(allpos.T), np.concatenate(types).astype(np.int32),
                       np.array(boxes))
