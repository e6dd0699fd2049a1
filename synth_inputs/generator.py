"""Seeded water-box generator (numpy only).

Draw order is fixed (documented per function) so that a given (recipe, seed)
always yields bit-identical arrays on every machine: all draws come from
``numpy.random.Generator(numpy.random.PCG64(seed))``.

Units: Angstrom, elementary charge, Angstrom^3 (polarizability).
Quadrupoles are traceless Cartesian (Buckingham) tensors stored as the six
unique components (xx, xy, xz, yy, yz, zz).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
import math

import numpy as np

# rigid water geometry, BASELINE.json configs[0]
_OH = 0.9572
_HOH = math.radians(104.52)
_Q_O, _Q_H = -0.51966, 0.25983
_POL_O, _POL_H = 0.837, 0.496
THOLE_A = 0.39


@dataclass
class System:
    """One synthetic system; arrays are C-contiguous float64 / int32."""
    name: str
    box: float                 # cubic edge (A); <= 0 means open boundary
    pos: np.ndarray            # (N,3), molecules kept whole (NOT wrapped)
    charge: np.ndarray         # (N,)
    dipole: np.ndarray         # (N,3)
    quad: np.ndarray           # (N,6) xx,xy,xz,yy,yz,zz ; traceless
    polarizability: np.ndarray  # (N,)
    group_id: np.ndarray       # (N,) int32 polarization group (= molecule)
    cutoff: float = 7.0
    skin: float = 2.0
    ewald_beta: float = 0.5446
    thole_a: float = THOLE_A
    seed: int = 0
    meta: dict = field(default_factory=dict)

    @property
    def n_atoms(self) -> int:
        return int(self.pos.shape[0])

    def with_(self, **kw) -> "System":
        return replace(self, **kw)


def beta_for_cutoff(cutoff: float) -> float:
    """keep beta*rc at BASELINE's 7 A value (0.5446*7)."""
    return 0.5446 * 7.0 / cutoff


def _random_rotations(rng: np.random.Generator, m: int) -> np.ndarray:
    """m rotation matrices from normalised 4-Gaussian quaternions."""
    q = rng.standard_normal((m, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    rot = np.empty((m, 3, 3))
    rot[:, 0, 0] = 1 - 2 * (y * y + z * z)
    rot[:, 0, 1] = 2 * (x * y - z * w)
    rot[:, 0, 2] = 2 * (x * z + y * w)
    rot[:, 1, 0] = 2 * (x * y + z * w)
    rot[:, 1, 1] = 1 - 2 * (x * x + z * z)
    rot[:, 1, 2] = 2 * (y * z - x * w)
    rot[:, 2, 0] = 2 * (x * z - y * w)
    rot[:, 2, 1] = 2 * (y * z + x * w)
    rot[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return rot


def _traceless_quads(rng: np.random.Generator, n: int, sigma: float) -> np.ndarray:
    a = rng.standard_normal((n, 3, 3)) * sigma
    s = 0.5 * (a + a.transpose(0, 2, 1))
    tr = (s[:, 0, 0] + s[:, 1, 1] + s[:, 2, 2]) / 3.0
    for k in range(3):
        s[:, k, k] -= tr
    return np.stack([s[:, 0, 0], s[:, 0, 1], s[:, 0, 2],
                     s[:, 1, 1], s[:, 1, 2], s[:, 2, 2]], axis=1)


def _min_image(d: np.ndarray, box: float) -> np.ndarray:
    return d - box * np.round(d / box) if box > 0 else d


def water_box(n_mol: int, box: float, seed: int, *, solute_frac: float = 0.0,
              cutoff: float = 7.0, skin: float = 2.0, ewald_beta: float = 0.5446,
              name: str = "water") -> System:
    """Jittered-lattice rigid water box (SURVEY 8(d) geometry recipe).

    Draw order: (1) lattice-site choice, (2) O jitter, (3) quaternions,
    (4) dipoles, (5) quadrupoles, then for solutes (6) molecule choice and,
    per redraw round, (7) directions, (8) radii; finally (9) solute charges,
    (10) solute dipoles, (11) solute quadrupoles, (12) solute polarizabilities.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    n_lat = int(math.ceil(n_mol ** (1.0 / 3.0) - 1e-9))
    while n_lat ** 3 < n_mol:
        n_lat += 1
    sites = n_lat ** 3
    if n_mol < sites:
        chosen = np.sort(rng.choice(sites, size=n_mol, replace=False))
    else:
        chosen = np.arange(sites)
    ix = chosen // (n_lat * n_lat)
    iy = (chosen // n_lat) % n_lat
    iz = chosen % n_lat
    h = box / n_lat
    centre = (np.stack([ix, iy, iz], axis=1) + 0.5) * h
    centre = centre + rng.uniform(-0.25, 0.25, size=(n_mol, 3))
    rot = _random_rotations(rng, n_mol)
    local = np.array([[0.0, 0.0, 0.0],
                      [_OH * math.sin(_HOH / 2), 0.0, _OH * math.cos(_HOH / 2)],
                      [-_OH * math.sin(_HOH / 2), 0.0, _OH * math.cos(_HOH / 2)]])
    pos = centre[:, None, :] + np.einsum("mab,kb->mka", rot, local)
    n = 3 * n_mol
    pos = pos.reshape(n, 3)
    charge = np.tile([_Q_O, _Q_H, _Q_H], n_mol).astype(np.float64)
    alpha = np.tile([_POL_O, _POL_H, _POL_H], n_mol).astype(np.float64)
    dipole = rng.standard_normal((n, 3)) * 0.1
    quad = _traceless_quads(rng, n, 0.1)
    group = np.repeat(np.arange(n_mol, dtype=np.int32), 3)
    meta = {"n_mol": n_mol, "n_lattice": n_lat, "n_solute": 0}

    n_sol = int(round(solute_frac * n_mol))
    if n_sol > 0:
        from scipy.spatial import cKDTree
        sol = np.sort(rng.choice(n_mol, size=n_sol, replace=False))
        todo = sol.copy()
        rounds = 0
        while todo.size:
            rounds += 1
            if rounds > 200:
                raise RuntimeError("solute placement did not converge")
            k = todo.size
            v = rng.standard_normal((k, 3, 3))
            v /= np.linalg.norm(v, axis=2, keepdims=True)
            rad = rng.uniform(0.6, 1.2, size=(k, 3))
            newp = centre[todo][:, None, :] + v * rad[:, :, None]
            pos.reshape(n_mol, 3, 3)[todo] = newp
            # intra-group site spacing >= 1.0 A
            p = pos.reshape(n_mol, 3, 3)[sol]
            d01 = np.linalg.norm(p[:, 0] - p[:, 1], axis=1)
            d02 = np.linalg.norm(p[:, 0] - p[:, 2], axis=1)
            d12 = np.linalg.norm(p[:, 1] - p[:, 2], axis=1)
            bad = set(sol[(d01 < 1.0) | (d02 < 1.0) | (d12 < 1.0)].tolist())
            # >= 1.0 A from every atom of any other group (periodic)
            wrapped = pos - box * np.floor(pos / box)
            wrapped = np.minimum(wrapped, np.nextafter(box, 0.0))
            tree = cKDTree(wrapped, boxsize=box)
            close = tree.query_pairs(1.0, output_type="ndarray")
            is_sol = np.zeros(n_mol, dtype=bool)
            is_sol[sol] = True
            if close.size:
                ga, gb = group[close[:, 0]], group[close[:, 1]]
                inter = ga != gb
                for g in np.concatenate([ga[inter & is_sol[ga]], gb[inter & is_sol[gb]]]):
                    bad.add(int(g))
            todo = np.array(sorted(bad), dtype=np.int64)
        atoms = (sol[:, None] * 3 + np.arange(3)[None, :]).reshape(-1)
        charge[atoms] = rng.uniform(-0.8, 0.8, size=atoms.size)
        dipole[atoms] = rng.standard_normal((atoms.size, 3)) * 0.3
        quad[atoms] = _traceless_quads(rng, atoms.size, 0.3)
        alpha[atoms] = rng.uniform(0.3, 1.8, size=atoms.size)
        meta.update(n_solute=n_sol, solute_rounds=rounds)

    return System(name=name, box=float(box), pos=np.ascontiguousarray(pos),
                  charge=charge, dipole=np.ascontiguousarray(dipole),
                  quad=np.ascontiguousarray(quad), polarizability=alpha,
                  group_id=group, cutoff=cutoff, skin=skin, ewald_beta=ewald_beta,
                  thole_a=THOLE_A, seed=seed, meta=meta)


def tiny_cluster(n_atoms: int, seed: int, *, box: float = 0.0, spread: float = 4.0,
                 group_size: int = 3, cutoff: float = 7.0, skin: float = 2.0,
                 ewald_beta: float = 0.0, min_dist: float = 0.9) -> System:
    """Small random point cloud (tests: N = 2, 3, 33, 65 ...), open or periodic.

    Draw order: positions (rejection on ``min_dist``), charges, dipoles,
    quadrupoles, polarizabilities.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    pts: list[np.ndarray] = []
    while len(pts) < n_atoms:
        c = rng.uniform(0.0, spread, size=3)
        ok = True
        for p in pts:
            if np.linalg.norm(_min_image(c - p, box)) < min_dist:
                ok = False
                break
        if ok:
            pts.append(c)
    pos = np.array(pts).reshape(n_atoms, 3)
    charge = rng.uniform(-0.8, 0.8, size=n_atoms)
    dipole = rng.standard_normal((n_atoms, 3)) * 0.3
    quad = _traceless_quads(rng, n_atoms, 0.3)
    alpha = rng.uniform(0.3, 1.8, size=n_atoms)
    group = (np.arange(n_atoms) // group_size).astype(np.int32)
    return System(name=f"tiny{n_atoms}", box=float(box), pos=pos, charge=charge,
                  dipole=dipole, quad=quad, polarizability=alpha, group_id=group,
                  cutoff=cutoff, skin=skin, ewald_beta=ewald_beta, thole_a=THOLE_A,
                  seed=seed, meta={})


# BASELINE.json configs (index -> recipe); seeds per SURVEY 8(d).
CONFIGS = {
    0: dict(name="cfg0_water648", n_mol=216, box=18.64, seed=120700, solute_frac=0.0),
    1: dict(name="cfg1_dhfr_size", n_mol=7853, box=61.7, seed=120701, solute_frac=0.0),
    2: dict(name="cfg2_hetero98k", n_mol=32768, box=99.4, seed=120702, solute_frac=0.15),
    3: dict(name="cfg3_stmv_size", n_mol=355543, box=220.1, seed=120703, solute_frac=0.0),
}


def make_config(idx: int, *, cutoff: float = 7.0, skin: float = 2.0,
                ewald_beta: float | None = None) -> System:
    """BASELINE.json configs[idx]; config 4 is config 2 with another cutoff."""
    base = 2 if idx == 4 else idx
    c = CONFIGS[base]
    beta = beta_for_cutoff(cutoff) if ewald_beta is None else ewald_beta
    if abs(cutoff - 7.0) < 1e-12 and ewald_beta is None:
        beta = 0.5446
    return water_box(c["n_mol"], c["box"], c["seed"], solute_frac=c["solute_frac"],
                     cutoff=cutoff, skin=skin, ewald_beta=beta, name=c["name"])
