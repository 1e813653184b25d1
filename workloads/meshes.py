"""Cell-type meshes and the paper's material table (input generation only).

Units everywhere: micrometre, microsecond, femtogram, piconewton
(1 fg*um/us^2 = 1 pN), the self-consistent system implied by the parameter
table PAPER.md:226-239.

Rest shapes (SURVEY.md reading R14, BASELINE.json configs):
  * RBC: unit icosphere mapped through the Evans-Fung biconcave profile,
    radius R0 = 3.91 um ("normal biconcave").
  * platelet: unit icosphere scaled to an oblate ellipsoid with semi-axes
    (1.8, 1.8, 0.5) um (diameter 3.6 um, 6.8 fL).
Icospheres use midpoint subdivision with re-normalisation to the unit
sphere: V = 10*4^L + 2, T = 20*4^L, E = 30*4^L.
"""
from __future__ import annotations

import dataclasses
import itertools

import numpy as np


@dataclasses.dataclass(frozen=True)
class Material:
    """Material constants of one cell type."""

    skalak_B: float = 5.0          # pN/um
    skalak_C: float = 5000.0       # pN/um
    skalak_D: float = 35.0         # pN/um   PAPER.md:231 (carried, unused: reading R6)
    k_bending: float = 1.0         # pN*um
    k_volume: float = 250.0        # pN/um^2 PAPER.md:233 (unit is reading R9)
    rayleigh_alpha: float = 0.0    # 1/us
    rayleigh_beta: float = 0.01    # us
    kappa_damping: float = 0.5     # [0,1]   PAPER.md:235 (first listed value, reading R12)
    density: float = 1025.0        # fg/um^3 PAPER.md:239

    def scaled_stiffness(self, factor: float) -> "Material":
        """Same material with B, C, D, k_bending, k_volume multiplied by `factor`."""
        return dataclasses.replace(
            self,
            skalak_B=self.skalak_B * factor,
            skalak_C=self.skalak_C * factor,
            skalak_D=self.skalak_D * factor,
            k_bending=self.k_bending * factor,
            k_volume=self.k_volume * factor,
        )


@dataclasses.dataclass(frozen=True)
class CellType:
    """One cell type: closed, outward-oriented triangulated rest shape + material."""

    name: str
    rest_positions: np.ndarray  # [n, 3] float64
    triangles: np.ndarray       # [T, 3] int32, counter-clockwise seen from outside
    material: Material

    @property
    def n_vertices(self) -> int:
        return int(self.rest_positions.shape[0])

    @property
    def n_triangles(self) -> int:
        return int(self.triangles.shape[0])


def rbc_material() -> Material:
    """Red-blood-cell constants exactly as listed in PAPER.md:231-235."""
    return Material()


def platelet_material() -> Material:
    """Platelets are 'nearly-rigid bodies by increasing the stiffness'.

    Reading R13 (unpinned): ten times the RBC stiffness constants.
    """
    return Material().scaled_stiffness(10.0)


def icosahedron() -> tuple[np.ndarray, np.ndarray]:
    """Unit-circumradius icosahedron: 12 vertices, 20 outward CCW faces."""
    phi = (1.0 + np.sqrt(5.0)) / 2.0
    verts = []
    for s1 in (-1.0, 1.0):
        for s2 in (-1.0, 1.0):
            verts.append((0.0, s1, s2 * phi))
            verts.append((s1, s2 * phi, 0.0))
            verts.append((s2 * phi, 0.0, s1))
    v = np.array(sorted(set(verts)), dtype=np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    # faces = triples of mutually nearest vertices (edge length is the minimum distance)
    dist = np.linalg.norm(v[:, None, :] - v[None, :, :], axis=2)
    edge = np.min(dist[dist > 1e-9])
    adj = np.abs(dist - edge) < 1e-9
    faces = []
    for a, b, c in itertools.combinations(range(12), 3):
        if adj[a, b] and adj[b, c] and adj[a, c]:
            nrm = np.cross(v[b] - v[a], v[c] - v[a])
            if np.dot(nrm, v[a] + v[b] + v[c]) < 0.0:
                b, c = c, b
            faces.append((a, b, c))
    f = np.array(faces, dtype=np.int32)
    assert f.shape == (20, 3)
    return v, f


def icosphere(level: int) -> tuple[np.ndarray, np.ndarray]:
    """Icosahedron subdivided `level` times, new vertices pushed onto the unit sphere."""
    v, f = icosahedron()
    verts = [tuple(p) for p in v]
    for _ in range(level):
        cache: dict[tuple[int, int], int] = {}

        def midpoint(a: int, b: int) -> int:
            key = (a, b) if a < b else (b, a)
            idx = cache.get(key)
            if idx is None:
                m = 0.5 * (np.asarray(verts[a]) + np.asarray(verts[b]))
                m /= np.linalg.norm(m)
                idx = len(verts)
                verts.append(tuple(m))
                cache[key] = idx
            return idx

        new_f = []
        for a, b, c in f:
            ab, bc, ca = midpoint(a, b), midpoint(b, c), midpoint(c, a)
            new_f += [(a, ab, ca), (b, bc, ab), (c, ca, bc), (ab, bc, ca)]
        f = np.array(new_f, dtype=np.int32)
    return np.array(verts, dtype=np.float64), f


def octasphere(level: int) -> tuple[np.ndarray, np.ndarray]:
    """Octahedron subdivided `level` times onto the unit sphere: V = 4*4^L + 2 (66 at L = 2, 258 at L = 3,
    the paper's platelet / RBC resolutions), T = 8*4^L."""
    verts = [(1.0, 0, 0), (-1.0, 0, 0), (0, 1.0, 0), (0, -1.0, 0), (0, 0, 1.0), (0, 0, -1.0)]
    f = np.array([(0, 2, 4), (2, 1, 4), (1, 3, 4), (3, 0, 4), (2, 0, 5), (1, 2, 5), (3, 1, 5), (0, 3, 5)], dtype=np.int32)
    for _ in range(level):
        cache: dict[tuple[int, int], int] = {}

        def midpoint(a: int, b: int) -> int:
            key = (a, b) if a < b else (b, a)
            idx = cache.get(key)
            if idx is None:
                m = 0.5 * (np.asarray(verts[a], dtype=np.float64) + np.asarray(verts[b], dtype=np.float64))
                m /= np.linalg.norm(m)
                idx = len(verts)
                verts.append(tuple(m))
                cache[key] = idx
            return idx

        new_f = []
        for a, b, c in f:
            ab, bc, ca = midpoint(a, b), midpoint(b, c), midpoint(c, a)
            new_f += [(a, ab, ca), (b, bc, ab), (c, ca, bc), (ab, bc, ca)]
        f = np.array(new_f, dtype=np.int32)
    return np.array(verts, dtype=np.float64), f


# Evans-Fung biconcave profile constants (literature values, not in PAPER.md; reading R14)
_EF_C0, _EF_C1, _EF_C2 = 0.207161, 2.002558, -1.122762
RBC_RADIUS_UM = 3.91


def evans_fung_map(unit_points: np.ndarray, radius: float = RBC_RADIUS_UM) -> np.ndarray:
    """Map unit-sphere points (X,Y,Z) to (R0 X, R0 Y, sign(Z) z(r)) with the Evans-Fung z(r)."""
    x = radius * unit_points[:, 0]
    y = radius * unit_points[:, 1]
    rho2 = np.clip(unit_points[:, 0] ** 2 + unit_points[:, 1] ** 2, 0.0, 1.0)
    half = 0.5 * radius * np.sqrt(1.0 - rho2) * (_EF_C0 + _EF_C1 * rho2 + _EF_C2 * rho2 ** 2)
    z = np.sign(unit_points[:, 2]) * half
    return np.stack([x, y, z], axis=1)


def rbc_cell_type(level: int = 3, material: Material | None = None, base: str = "ico") -> CellType:
    v, f = icosphere(level) if base == "ico" else octasphere(level)
    return CellType(
        name=f"RBC-{v.shape[0]}",
        rest_positions=np.ascontiguousarray(evans_fung_map(v)),
        triangles=np.ascontiguousarray(f),
        material=material or rbc_material(),
    )


PLATELET_SEMI_AXES_UM = (1.8, 1.8, 0.5)


def platelet_cell_type(level: int = 2, material: Material | None = None, base: str = "ico") -> CellType:
    v, f = icosphere(level) if base == "ico" else octasphere(level)
    return CellType(
        name=f"PLT-{v.shape[0]}",
        rest_positions=np.ascontiguousarray(v * np.asarray(PLATELET_SEMI_AXES_UM)),
        triangles=np.ascontiguousarray(f),
        material=material or platelet_material(),
    )


def icosahedron_cell_type(circumradius: float = 3.0, material: Material | None = None) -> CellType:
    """The 12-vertex brute-force cell of the north star (SURVEY.md pins P8, P10)."""
    v, f = icosahedron()
    return CellType(
        name="ICO-12",
        rest_positions=np.ascontiguousarray(v * circumradius),
        triangles=np.ascontiguousarray(f),
        material=material or rbc_material(),
    )


def irregular_cell_type(level: int = 2, n_flips: int = 40, seed: int = 3, material: Material | None = None) -> CellType:
    """A closed mesh that is NOT an icosphere: interior edges of the platelet icosphere are flipped at
    random (valences spread over 4..8), so code that silently relies on valence <= 6 or on the
    subdivision ordering fails on it.  Edge-case input for the parity tests."""
    base = platelet_cell_type(level, material)
    rng = np.random.default_rng(seed)
    tri = [tuple(int(v) for v in t) for t in base.triangles]
    attempts = 0
    while n_flips > 0 and attempts < 100000:
        attempts += 1
        t = int(rng.integers(len(tri)))
        a, b, c = tri[t]
        other = next((i for i, u in enumerate(tri) if i != t and a in u and b in u), None)
        if other is None:
            continue
        d = next(v for v in tri[other] if v not in (a, b))
        val = np.bincount(np.array(tri).ravel(), minlength=base.n_vertices)
        if val[a] <= 4 or val[b] <= 4 or val[c] >= 8 or val[d] >= 8:
            continue
        if any(c in u and d in u for u in tri):
            continue
        # the flipped pair must stay convex enough to keep positive areas and outward orientation
        p = base.rest_positions
        n1 = np.cross(p[d] - p[a], p[c] - p[a])
        n2 = np.cross(p[b] - p[d], p[c] - p[d])
        if np.dot(n1, p[a] + p[d] + p[c]) <= 0 or np.dot(n2, p[d] + p[b] + p[c]) <= 0:
            continue
        if min(np.linalg.norm(n1), np.linalg.norm(n2)) < 0.2 * max(np.linalg.norm(n1), np.linalg.norm(n2)):
            continue
        if np.dot(n1, n2) < 0.9 * np.linalg.norm(n1) * np.linalg.norm(n2):      # keep the surface smooth
            continue
        tri[t], tri[other] = (a, d, c), (d, b, c)
        n_flips -= 1
    return CellType(name=f"IRR-{base.n_vertices}", rest_positions=base.rest_positions,
                    triangles=np.array(tri, dtype=np.int32), material=base.material)
