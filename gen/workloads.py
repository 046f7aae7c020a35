"""Seeded generators for configs C1..C5 (BASELINE.json:configs[0..4]; recipe in
SURVEY.md §8(d) and DESIGN.md §4).

Everything here is input synthesis: random draws, rejection of unlucky
geometries, dtype casts.  No symmetry function, cutoff function, gradient or
network is evaluated here -- those live in `oracle/` (fp64 CPU) and in the CUDA
library, which share no code.

All positions, box edges, parameters and upstream gradients are emitted as
float32: both sides consume the same float32 values, the
oracle promoting them to double.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, List, Optional, Tuple

import numpy as np
from scipy.spatial import cKDTree

MARGIN = 1.0e-4          # BASELINE.json:north_star "reject any distance within 1e-4 A of a cutoff"
COLLINEAR_EPS = 1.0e-7   # reject triplets with 1-|cos(theta)| < 1e-7


# --------------------------------------------------------------------------- parameters
@dataclasses.dataclass(frozen=True)
class AniParams:
    """ANI-1x-style AEV parameters (BASELINE.json:configs[0]); all float32."""
    num_species: int
    rcr: np.float32
    rca: np.float32
    eta_r: np.float32
    shf_r: np.ndarray      # float32 [n_shf_r]
    eta_a: np.float32
    zeta: np.float32
    shf_a: np.ndarray      # float32 [n_shf_a]
    shf_z: np.ndarray      # float32 [n_shf_z]
    cos_scale: np.float32  # 1.0 = literal north_star formula; 0.95 = damped variant (G2)

    @property
    def radial_length(self) -> int:
        return self.num_species * len(self.shf_r)

    @property
    def angular_length(self) -> int:
        s = self.num_species
        return s * (s + 1) // 2 * len(self.shf_a) * len(self.shf_z)

    @property
    def aev_length(self) -> int:
        return self.radial_length + self.angular_length


def ani1x_style_params(cos_scale: float = 1.0, num_species: int = 4, dtype=np.float32) -> AniParams:
    """Rcr=5.2, Rca=3.5; 16 radial shifts linspace(0.9,4.96875), eta_R=16; 4 angular
    radial shifts linspace(0.9,2.85), eta_A=8, zeta=32; 8 theta_s=(2k+1)pi/16
    (BASELINE.json:configs[0]; G8: endpoint included).  dtype=float32 is what every
    workload uses (G9); dtype=float64 gives the exact decimal parameters the closed-form
    fixtures in tests/golden/ were computed with."""
    t = np.dtype(dtype).type
    return AniParams(
        num_species=num_species,
        rcr=t(5.2),
        rca=t(3.5),
        eta_r=t(16.0),
        shf_r=np.linspace(0.9, 4.96875, 16).astype(dtype),
        eta_a=t(8.0),
        zeta=t(32.0),
        shf_a=np.linspace(0.9, 2.85, 4).astype(dtype),
        shf_z=((2.0 * np.arange(8) + 1.0) * math.pi / 16.0).astype(dtype),
        cos_scale=t(cos_scale),
    )


def ani2x_shaped_params(cos_scale: float = 1.0, num_species: int = 7) -> AniParams:
    """The OTHER angular split the library supports - 8 angular radial shifts x 4 angle shifts, a zeta that is not
    a power of two, 7 species (L = 1008) - with synthetic, evenly spaced shifts of this repository's own choosing
    (the same ranges as the ANI-1x-style set): the SHAPE of a 2x-generation parameter set, not its published values."""
    t = np.float32
    return AniParams(
        num_species=num_species,
        rcr=t(5.2),
        rca=t(3.5),
        eta_r=t(16.0),
        shf_r=np.linspace(0.9, 4.96875, 16).astype(np.float32),
        eta_a=t(8.0),
        zeta=t(14.1),
        shf_a=np.linspace(0.9, 2.85, 8).astype(np.float32),
        shf_z=((2.0 * np.arange(4) + 1.0) * math.pi / 8.0).astype(np.float32),
        cos_scale=t(cos_scale),
    )


@dataclasses.dataclass
class Workload:
    name: str
    pos: np.ndarray                 # float32 [batch, n_atoms, 3]
    species: np.ndarray             # int32   [batch, n_atoms]
    box: Optional[np.ndarray]       # float32 [3] or None (non-periodic)
    grad_aev: np.ndarray            # float32 [batch, n_atoms, L]   upstream dE/dAEV ~ N(0,1)
    params: AniParams

    @property
    def batch(self) -> int:
        return self.pos.shape[0]

    @property
    def n_atoms(self) -> int:
        return self.pos.shape[1]


# --------------------------------------------------------------------------- geometry checks
def _min_image(d: np.ndarray, box: Optional[np.ndarray]) -> np.ndarray:
    if box is None:
        return d
    b = box.astype(np.float64)
    return d - b * np.rint(d / b)


def _candidate_pairs(pos64: np.ndarray, box: Optional[np.ndarray], radius: float) -> np.ndarray:
    """Undirected candidate pairs (i<j) within `radius` (slightly padded by the caller)."""
    if box is None:
        tree = cKDTree(pos64)
    else:
        b = box.astype(np.float64)
        wrapped = pos64 - b * np.floor(pos64 / b)
        wrapped = np.where(wrapped >= b, wrapped - b, wrapped)
        wrapped = np.where(wrapped < 0.0, 0.0, wrapped)
        tree = cKDTree(wrapped, boxsize=b)
    return tree.query_pairs(radius, output_type="ndarray")


def _pair_distances(pos64, pairs, box):
    d = _min_image(pos64[pairs[:, 1]] - pos64[pairs[:, 0]], box)
    return np.sqrt((d * d).sum(axis=1)), d


def _bad_atoms(pos32: np.ndarray, box: Optional[np.ndarray], rcr: float, rca: float,
               min_dist: float = 0.0, mol_id: Optional[np.ndarray] = None) -> np.ndarray:
    """Atoms involved in (a) a pair within MARGIN of either cutoff, (b) a pair from
    different molecules closer than min_dist, (c) a near-collinear angular triplet."""
    pos64 = pos32.astype(np.float64)
    pairs = _candidate_pairs(pos64, box, rcr + 0.01)
    if len(pairs) == 0:
        return np.zeros(0, dtype=np.int64)
    r, d = _pair_distances(pos64, pairs, box)
    bad = (np.abs(r - rcr) < MARGIN) | (np.abs(r - rca) < MARGIN)
    if min_dist > 0.0:
        inter = np.ones(len(pairs), dtype=bool) if mol_id is None else (
            mol_id[pairs[:, 0]] != mol_id[pairs[:, 1]])
        bad |= inter & (r < min_dist)
    out = [pairs[bad].ravel()]
    # collinear triplets among angular neighbours
    ang = r < rca
    pi = np.concatenate([pairs[ang, 0], pairs[ang, 1]])
    pj = np.concatenate([pairs[ang, 1], pairs[ang, 0]])
    dv = np.concatenate([d[ang], -d[ang]])
    rv = np.concatenate([r[ang], r[ang]])
    order = np.argsort(pi, kind="stable")
    pi, pj, dv, rv = pi[order], pj[order], dv[order], rv[order]
    n = pos32.shape[0]
    cnt = np.bincount(pi, minlength=n)
    start = np.concatenate([[0], np.cumsum(cnt)])
    u = dv / rv[:, None]
    for c in np.unique(cnt):
        if c < 2:
            continue
        atoms = np.nonzero(cnt == c)[0]
        idx = start[atoms][:, None] + np.arange(c)[None, :]
        uu = u[idx]                                   # [m, c, 3]
        cs = np.einsum("mad,mbd->mab", uu, uu)
        iu = np.triu_indices(c, k=1)
        viol = (1.0 - np.abs(cs[:, iu[0], iu[1]])) < COLLINEAR_EPS
        if viol.any():
            m_idx, t_idx = np.nonzero(viol)
            out.append(atoms[m_idx])
            out.append(pj[idx[m_idx, iu[0][t_idx]]])
            out.append(pj[idx[m_idx, iu[1][t_idx]]])
    return np.unique(np.concatenate(out))


def _grad_aev(shape, seed: int = 0) -> np.ndarray:
    """Upstream dE/dAEV ~ N(0,1), seed 0 (BASELINE.json:configs[0])."""
    return np.random.default_rng(seed).standard_normal(shape).astype(np.float32)


# --------------------------------------------------------------------------- C1
def make_c1(cos_scale: float = 1.0) -> Workload:
    """24 atoms uniform in [0,6)^3 A, redrawn until every pair >= 0.9 A and the
    cutoff margins are clean; 10 H / 8 C / 3 N / 3 O; non-periodic
    (BASELINE.json:configs[0]; seeds: pos 100, species 101, g 0)."""
    p = ani1x_style_params(cos_scale)
    rng = np.random.default_rng(100)
    while True:
        pos = rng.uniform(0.0, 6.0, size=(24, 3)).astype(np.float32)
        p64 = pos.astype(np.float64)
        dd = p64[:, None, :] - p64[None, :, :]
        r = np.sqrt((dd * dd).sum(-1))[np.triu_indices(24, 1)]
        if r.min() < 0.9:
            continue
        if len(_bad_atoms(pos, None, float(p.rcr), float(p.rca))):
            continue
        break
    species = np.array([0] * 10 + [1] * 8 + [2] * 3 + [3] * 3, dtype=np.int32)
    np.random.default_rng(101).shuffle(species)
    return Workload("C1", pos[None], species[None], None,
                    _grad_aev((1, 24, p.aev_length)), p)


# --------------------------------------------------------------------------- C2
def _random_unit(rng) -> np.ndarray:
    v = rng.standard_normal(3)
    return v / np.linalg.norm(v)


def _ligand_conformer(rng, heavy: int = 32, hydrogens: int = 28) -> np.ndarray:
    """Self-avoiding random chain of `heavy` atoms (bond 1.4 + U(-0.1,0.1) A, non-bonded
    heavy atoms >= 2.0 A) plus `hydrogens` H at 1.0 A from heavy atoms taken
    round-robin, each rejected if < 1.3 A from any other atom."""
    while True:
        pts = [np.zeros(3)]
        stuck = False
        for a in range(1, heavy):
            for _ in range(200):
                cand = pts[-1] + (1.4 + rng.uniform(-0.1, 0.1)) * _random_unit(rng)
                if a >= 2:
                    prev = np.asarray(pts[:-1])
                    if np.sqrt(((prev - cand) ** 2).sum(1)).min() < 2.0:
                        continue
                pts.append(cand)
                break
            else:
                stuck = True
                break
        if stuck:
            continue
        atoms = list(pts)
        ok = True
        for h in range(hydrogens):
            parent = h % heavy
            for _ in range(400):
                cand = pts[parent] + 1.0 * _random_unit(rng)
                others = np.asarray(atoms)
                dist = np.sqrt(((others - cand) ** 2).sum(1))
                dist[parent] = np.inf
                if dist.min() < 1.3:
                    continue
                atoms.append(cand)
                break
            else:
                ok = False
                break
        if ok:
            return np.asarray(atoms)


def make_c2(cos_scale: float = 1.0, batch: int = 256) -> Workload:
    """256 conformers of a 60-atom ligand-like ML region (53-atom
    inhibitor), 28 H / 22 C / 5 N / 5 O, N(0,0.05) A jitter (BASELINE.json:configs[1];
    seeds: pos 200+conformer, species 201, g 0).  Atom order: 32 heavy, then 28 H."""
    p = ani1x_style_params(cos_scale)
    heavy_species = np.array([1] * 22 + [2] * 5 + [3] * 5, dtype=np.int32)
    np.random.default_rng(201).shuffle(heavy_species)
    species1 = np.concatenate([heavy_species, np.zeros(28, dtype=np.int32)])
    pos = np.empty((batch, 60, 3), dtype=np.float32)
    for c in range(batch):
        rng = np.random.default_rng(200 + c)
        base = _ligand_conformer(rng)
        while True:
            conf = (base + rng.normal(0.0, 0.05, size=base.shape)).astype(np.float32)
            if len(_bad_atoms(conf, None, float(p.rcr), float(p.rca))) == 0:
                break
        pos[c] = conf
    species = np.broadcast_to(species1, (batch, 60)).copy()
    return Workload("C2", pos, species, None, _grad_aev((batch, 60, p.aev_length)), p)


# --------------------------------------------------------------------------- C3 / C4
_OH = 0.9572
_HOH = math.radians(104.52)
_WATER = np.array([
    [0.0, 0.0, 0.0],
    [+_OH * math.sin(_HOH / 2), 0.0, _OH * math.cos(_HOH / 2)],
    [-_OH * math.sin(_HOH / 2), 0.0, _OH * math.cos(_HOH / 2)],
])


def _rotations(rng, m: int) -> np.ndarray:
    q = rng.standard_normal((m, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    rot = np.empty((m, 3, 3))
    rot[:, 0, 0] = 1 - 2 * (y * y + z * z); rot[:, 0, 1] = 2 * (x * y - z * w); rot[:, 0, 2] = 2 * (x * z + y * w)
    rot[:, 1, 0] = 2 * (x * y + z * w); rot[:, 1, 1] = 1 - 2 * (x * x + z * z); rot[:, 1, 2] = 2 * (y * z - x * w)
    rot[:, 2, 0] = 2 * (x * z - y * w); rot[:, 2, 1] = 2 * (y * z + x * w); rot[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return rot


def make_water_box(n_waters: int, side, seed: int, name: str,
                   cos_scale: float = 1.0) -> Workload:
    """Rigid waters (O-H 0.9572 A, HOH 104.52 deg) on a jittered partially filled
    lattice, random orientations, periodic box (BASELINE.json:configs[2,3]).  `side` is one
    edge length (cubic box, the recipe of C3/C4) or three (orthorhombic box, PAPER.md:223:
    the lattice then has ceil(L_k / (V/n)^(1/3)) sites along edge k).
    Atom order O,H,H per molecule; species O=3, H=0 (G7: S=4 everywhere).  Molecules are
    kept whole, so some H lie slightly outside [0,L) (G16)."""
    p = ani1x_style_params(cos_scale)
    rng = np.random.default_rng(seed)
    if np.ndim(side) == 0:
        n = int(math.ceil(n_waters ** (1.0 / 3.0) - 1e-9))
        nk = np.array([n, n, n])
        sides = np.array([float(side)] * 3)
    else:
        sides = np.asarray(side, dtype=np.float64).reshape(3)
        s0 = (sides.prod() / n_waters) ** (1.0 / 3.0)
        nk = np.ceil(sides / s0 - 1e-9).astype(np.int64)
    spacing = sides / nk
    sites = rng.permutation(int(nk.prod()))[:n_waters]
    ix, iy, iz = sites // (nk[1] * nk[2]), (sites // nk[2]) % nk[1], sites % nk[2]
    centre = (np.stack([ix, iy, iz], axis=1) + 0.5) * spacing

    def place(m):
        jit = rng.uniform(-0.25, 0.25, size=(m, 3))
        rot = _rotations(rng, m)
        return jit, np.einsum("mij,aj->mai", rot, _WATER)

    jit, rel = place(n_waters)
    box = sides.astype(np.float32)
    mol_id = np.repeat(np.arange(n_waters), 3)
    for _ in range(100):
        pos = ((centre + jit)[:, None, :] + rel).reshape(-1, 3).astype(np.float32)
        bad = _bad_atoms(pos, box, float(p.rcr), float(p.rca), min_dist=1.2, mol_id=mol_id)
        if len(bad) == 0:
            break
        mols = np.unique(mol_id[bad])
        j2, r2 = place(len(mols))
        jit[mols], rel[mols] = j2, r2
    else:
        raise RuntimeError("water box repair did not converge")
    species = np.tile(np.array([3, 0, 0], dtype=np.int32), n_waters)
    return Workload(name, pos[None], species[None], box,
                    _grad_aev((1, 3 * n_waters, p.aev_length)), p)


def make_c3(cos_scale: float = 1.0) -> Workload:
    """1,500 H2O, 4,500 atoms, L = 35.5 A (BASELINE.json:configs[2]; seed 300)."""
    return make_water_box(1500, 35.5, 300, "C3", cos_scale)


def make_c4(cos_scale: float = 1.0) -> Workload:
    """7,853 H2O, 23,559 atoms, L = 61.7 A -- DHFR-sized
    (BASELINE.json:configs[3]; seed 400)."""
    return make_water_box(7853, 61.7, 400, "C4", cos_scale)


# --------------------------------------------------------------------------- C5 weights
C5_ARCH: Dict[int, List[int]] = {
    0: [384, 160, 128, 96, 1],   # H
    3: [384, 128, 112, 96, 1],   # O
}
CELU_ALPHA = 0.1


def make_periodic_cell(n_atoms: int, cell, seed: int, name: str = "cell", cos_scale: float = 1.0,
                       min_dist: float = 1.1, params: Optional[AniParams] = None) -> Workload:
    """`n_atoms` atoms of species H/C/N/O (uniform) at random positions in a small periodic cell
    (the ML region can itself be a periodic cell of a few hundred atoms).  `cell` is three
    edge lengths (orthorhombic) or a 3x3 matrix of lattice rows a, b, c (triclinic, reduced form).
    Atoms are drawn one by one in fractional coordinates and rejected if closer than `min_dist` to an
    earlier atom or within MARGIN of a cutoff (distances over the 27 nearest images, float64); a third of
    the atoms is then moved by whole lattice vectors so that positions lie outside the cell.
    `Workload.box` is float32 [3] or [9] (lattice rows); `cell` None = a non-periodic cluster drawn in a 14 A cube.
    `params` (default: the ANI-1x-style set) fixes the cutoffs of the margin test and the species count."""
    p = ani1x_style_params(cos_scale) if params is None else params
    periodic = cell is not None
    if not periodic:
        cell = [14.0, 14.0, 14.0]
    rng = np.random.default_rng(seed)
    cell = np.asarray(cell, dtype=np.float64)
    lat = np.diag(cell) if cell.size == 3 else cell.reshape(3, 3)
    lat = lat.astype(np.float32).astype(np.float64)
    shifts = np.array([[i, j, k] for i in (-1, 0, 1) for j in (-1, 0, 1) for k in (-1, 0, 1)], dtype=np.float64) @ lat
    if not periodic:
        shifts = np.zeros((1, 3))
    pos = np.zeros((0, 3))
    rcr, rca = float(p.rcr), float(p.rca)
    tries = 0
    while len(pos) < n_atoms:
        tries += 1
        if tries > 200 * n_atoms:
            raise RuntimeError("periodic cell generator did not converge")
        x = (rng.random(3) @ lat).astype(np.float32).astype(np.float64)
        if len(pos):
            d = (pos[:, None, :] - x[None, None, :]) + shifts[None, :, :]
            r = np.sqrt((d * d).sum(axis=2)).min(axis=1)
            if r.min() < min_dist or (np.abs(r - rcr) < 10 * MARGIN).any() or (np.abs(r - rca) < 10 * MARGIN).any():
                continue
        pos = np.vstack([pos, x])
    if periodic:
        move = rng.random(n_atoms) < 0.33
        pos = pos + np.where(move[:, None], rng.integers(-2, 3, size=(n_atoms, 3)).astype(np.float64) @ lat, 0.0)
    species = rng.integers(0, int(p.num_species), size=n_atoms).astype(np.int32)
    box = None if not periodic else (cell if cell.size == 3 else lat.reshape(9)).astype(np.float32)
    return Workload(name, pos.astype(np.float32)[None], species[None], box,
                    _grad_aev((1, n_atoms, p.aev_length), seed), p)


def random_walk(w: Workload, n_steps: int, sigma: float, seed: int) -> List[np.ndarray]:
    """MD-like trajectory for the neighbour-list reuse tests (10,000 consecutive steps): every step adds
    N(0, sigma) to every coordinate; atoms that end up within MARGIN of a cutoff (or nearly collinear) get a new
    draw, so that every frame keeps the generators' guarantee.  Returns n_steps float32 arrays shaped like w.pos."""
    rng = np.random.default_rng(seed)
    frames = []
    cur = w.pos.astype(np.float64)
    p = w.params
    for _ in range(n_steps):
        step = rng.normal(0.0, sigma, size=cur.shape)
        for _try in range(50):
            new = (cur + step).astype(np.float32)
            bad_any = False
            for b in range(new.shape[0]):
                bad = _bad_atoms(new[b], w.box, float(p.rcr), float(p.rca))
                if len(bad):
                    bad_any = True
                    step[b, bad] = rng.normal(0.0, sigma, size=(len(bad), 3))
            if not bad_any:
                break
        else:
            raise RuntimeError("random walk repair did not converge")
        frames.append(new)
        cur = new.astype(np.float64)
    return frames


def _round_to_bf16(x: np.ndarray) -> np.ndarray:
    """Round float32 to the nearest bf16-representable float32 (ties to even)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32)


def make_c5_weights(seed: int = 1, arch: Optional[Dict[int, List[int]]] = None, round_bf16: bool = True
                    ) -> Dict[int, Tuple[List[np.ndarray], List[np.ndarray]]]:
    """Random-init per-species MLPs (BASELINE.json:configs[4]): weights and biases
    ~ N(0, 1/fan_in) (variance; G13), draw order species H then O, layer 0..3, W then b,
    one default_rng(seed) stream.  W is [in][out] row-major float32, rounded to
    bf16-representable values, which DEFINES the model (G14); biases stay float32.
    round_bf16=False keeps the float32 draws (a "trained-like" network whose weights are not
    bf16-representable)."""
    arch = C5_ARCH if arch is None else arch
    rng = np.random.default_rng(seed)
    out = {}
    for s in sorted(arch):
        dims = arch[s]
        ws, bs = [], []
        for l in range(len(dims) - 1):
            std = dims[l] ** -0.5
            w = (rng.standard_normal((dims[l], dims[l + 1])) * std).astype(np.float32)
            b = (rng.standard_normal(dims[l + 1]) * std).astype(np.float32)
            ws.append(_round_to_bf16(w) if round_bf16 else w)
            bs.append(b)
        out[s] = (ws, bs)
    return out


def make_ensemble_weights(n_models: int = 8, arch: Optional[Dict[int, List[int]]] = None, round_bf16: bool = True):
    """An ensemble of `n_models` independently initialised networks per species (ANI-2x is
    an ensemble of eight models): model m is make_c5_weights(seed = 1 + m)."""
    return [make_c5_weights(seed=1 + m, arch=arch, round_bf16=round_bf16) for m in range(n_models)]


# --------------------------------------------------------------------------- registry
_CACHE: Dict[Tuple[str, float], Workload] = {}


def make_workload(name: str, cos_scale: float = 1.0) -> Workload:
    key = (name.upper(), float(cos_scale))
    if key not in _CACHE:
        fn = {"C1": make_c1, "C2": make_c2, "C3": make_c3, "C4": make_c4, "C5": make_c3}[key[0]]
        _CACHE[key] = fn(cos_scale)
    return _CACHE[key]
