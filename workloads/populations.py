"""Seeded synthetic cell populations for the five BASELINE.json configs.

The paper measures on its own coupled simulations (Table 1);
there is no public dataset.  These populations take the SHAPE of that
workload (RBC + platelet mixes at 35 % hematocrit, random placement with
interpenetration allowed PAPER.md:79, shear-like forcing along one axis) and
stand in for it.  Recipe: SURVEY.md section 8(d), restated in DESIGN.md.

All draws use numpy.random.Generator(PCG64) child streams spawned from one
SeedSequence per config, in fp64.  "N(0, s)" means iid per Cartesian
component with standard deviation s.  No solver arithmetic lives here.
"""
from __future__ import annotations

import dataclasses

import numpy as np

from .meshes import CellType, platelet_cell_type, rbc_cell_type

CONFIG_NAMES = {
    1: "single RBC-642, N(0,1 pN) forces, 1 step x 10 its, dt 0.1 us",
    2: "1,000 RBC-642, random rigid placements, N(0,1 pN) forces, 10 steps x 10 its",
    3: "20,000 RBC-642 + 2,000 PLT-162 at 35% Hct, shear-like forces, 20 steps x 5 its",
    4: "90,000 RBC-642 + 10,000 PLT-162, shear-like forces, 10 steps x 10 its",
    5: "10,000 RBC-2562, N(0,1 pN) forces, 10 steps x K its",
    6: "the paper's own per-GPU load: 95 RBC-258 + 19 PLT-66 (octahedral meshes), h = 0.25 us, shear-like forces, "
       "20 steps x 5 its",
}


def _haar_rotations(rng: np.random.Generator, count: int) -> np.ndarray:
    """Haar-uniform rotation matrices from normalised 4-Gaussian quaternions."""
    q = rng.standard_normal((count, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    rot = np.empty((count, 3, 3))
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


@dataclasses.dataclass
class Population:
    """A batch of cells, bucketed by type.  Per-type arrays are [cells_t, n_t, 3] fp64."""

    name: str
    types: list[CellType]
    type_of_cell: np.ndarray                 # [n_cells] int32
    positions: list[np.ndarray]              # per type
    velocities: list[np.ndarray]             # per type
    dt: float                                # us
    n_steps: int
    n_iterations: int
    box: tuple[float, float, float]          # um
    force_sigma: float                       # pN
    shear_gamma: float                       # pN/um (0 = no shear term)
    redraw_noise_each_step: bool
    _force_seed: np.random.SeedSequence = None
    _shear_height: list[np.ndarray] = None   # per type [cells_t, n_t], z above mid-plane at t=0
    _const_forces: list[np.ndarray] = None

    @property
    def n_cells(self) -> int:
        return int(self.type_of_cell.shape[0])

    def cells_of_type(self, t: int) -> np.ndarray:
        """Cell ids of type t in bucket (ascending id) order."""
        return np.nonzero(self.type_of_cell == t)[0].astype(np.int64)

    # ---- forces -------------------------------------------------------------------------
    def _draw_forces(self, step: int) -> list[np.ndarray]:
        out = []
        for t, pos in enumerate(self.positions):
            # stateless child stream per (step, type): same values however often it is asked for
            child = np.random.SeedSequence(entropy=self._force_seed.entropy,
                                           spawn_key=self._force_seed.spawn_key + (step, t))
            rng = np.random.Generator(np.random.PCG64(child))
            f = self.force_sigma * rng.standard_normal(pos.shape)
            if self.shear_gamma != 0.0:
                f[..., 0] += self.shear_gamma * self._shear_height[t]
            out.append(f)
        return out

    def forces(self, step: int = 0) -> list[np.ndarray]:
        """External forces F_ext (pN) applied during time step `step`, per type."""
        if self.redraw_noise_each_step:
            return self._draw_forces(step)
        if self._const_forces is None:
            self._const_forces = self._draw_forces(0)
        return self._const_forces

    # ---- packing for the C-ABI: cells in `cell_ids` order, each [n_t][3] ----------------
    def vertex_counts(self) -> np.ndarray:
        n_of_type = np.array([ct.n_vertices for ct in self.types], dtype=np.int64)
        return n_of_type[self.type_of_cell]

    def packed(self, per_type: list[np.ndarray], cell_ids: np.ndarray | None = None,
               dtype=np.float64) -> np.ndarray:
        """Flatten a per-type field to one buffer: listed cells back to back, each [n][3]."""
        counts = self.vertex_counts()
        slot = np.zeros(self.n_cells, dtype=np.int64)
        for t in range(len(self.types)):
            ids = self.cells_of_type(t)
            slot[ids] = np.arange(ids.shape[0])
        if cell_ids is None:
            cell_ids = np.arange(self.n_cells, dtype=np.int64)
        sizes = 3 * counts[cell_ids]
        offsets = np.concatenate([[0], np.cumsum(sizes)])
        out = np.empty(int(offsets[-1]), dtype=dtype)
        for t, arr in enumerate(per_type):
            sel = np.nonzero(self.type_of_cell[cell_ids] == t)[0]
            if sel.size == 0:
                continue
            width = 3 * self.types[t].n_vertices
            dest = offsets[sel][:, None] + np.arange(width)[None, :]
            out[dest] = arr[slot[cell_ids[sel]]].reshape(sel.size, width)
        return out

    def unpack(self, flat: np.ndarray, cell_ids: np.ndarray | None = None) -> list[np.ndarray]:
        """Inverse of `packed` for a full or partial id list: per-type [k_t, n_t, 3] in list order."""
        counts = self.vertex_counts()
        if cell_ids is None:
            cell_ids = np.arange(self.n_cells, dtype=np.int64)
        sizes = 3 * counts[cell_ids]
        offsets = np.concatenate([[0], np.cumsum(sizes)])
        out = []
        for t, ct in enumerate(self.types):
            sel = np.nonzero(self.type_of_cell[cell_ids] == t)[0]
            width = 3 * ct.n_vertices
            src = offsets[sel][:, None] + np.arange(width)[None, :]
            out.append(np.asarray(flat)[src].reshape(sel.size, ct.n_vertices, 3))
        return out

    def subset(self, cell_ids: np.ndarray) -> "Population":
        """The listed cells as their own population (cells are independent: PAPER.md:61,63)."""
        cell_ids = np.asarray(cell_ids, dtype=np.int64)
        slot = np.zeros(self.n_cells, dtype=np.int64)
        for t in range(len(self.types)):
            ids = self.cells_of_type(t)
            slot[ids] = np.arange(ids.shape[0])
        order = np.sort(cell_ids)
        pos, vel, height, sel_slots = [], [], [], []
        for t in range(len(self.types)):
            s = slot[order[self.type_of_cell[order] == t]]
            sel_slots.append(s)
            pos.append(self.positions[t][s])
            vel.append(self.velocities[t][s])
            height.append(None if self._shear_height is None else self._shear_height[t][s])
        parent = self

        sub = Population(
            name=self.name + f" [subset of {order.size}]", types=self.types,
            type_of_cell=self.type_of_cell[order].copy(), positions=pos, velocities=vel,
            dt=self.dt, n_steps=self.n_steps, n_iterations=self.n_iterations, box=self.box,
            force_sigma=self.force_sigma, shear_gamma=self.shear_gamma,
            redraw_noise_each_step=self.redraw_noise_each_step,
            _force_seed=self._force_seed, _shear_height=height)
        # forces of a subset are the parent's forces restricted to the subset (same values)
        sub.forces = lambda step=0: [f[s] for f, s in zip(parent.forces(step), sel_slots)]  # type: ignore
        sub.parent_ids = order  # type: ignore
        return sub


def make_config(index: int, n_cells: int | None = None, level: int | None = None) -> Population:
    """Build BASELINE.json config `index` (1..5); `n_cells` shrinks it, keeping the recipe.
    Index 6 is not a BASELINE config: the paper's own resolutions and per-GPU load:
    RBC 258 / platelet 66 surface vertices, PLT:RBC = 1:5, 571 cells of the 50^3 um^3
    domain over 5 GPU nodes = 114 cells per GPU, solid step = 2 LBM steps = 0.25 us
    (PAPER.md:45, :230)."""
    if index not in CONFIG_NAMES:
        raise ValueError(f"config index must be 1..6, got {index}")
    seed = np.random.SeedSequence(index - 1)          # seeds 0..4
    s_rot, s_trans, s_force = seed.spawn(3)
    dt = 0.1                                           # 1e-7 s
    sigma, gamma, redraw = 1.0, 0.0, False
    if index == 1:
        total, period, box, steps, its = 1, 0, (0.0, 0.0, 0.0), 1, 10
        types = [rbc_cell_type(level if level is not None else 3)]
    elif index == 2:
        total, period, box, steps, its = 1000, 0, (50.0, 100.0, 50.0), 10, 10
        types = [rbc_cell_type(level if level is not None else 3)]
    elif index == 3:
        total, period, box, steps, its = 22000, 11, (175.0,) * 3, 20, 5
        types = [rbc_cell_type(3), platelet_cell_type(2)]
        sigma, gamma, redraw = 0.2, 0.02, True
    elif index == 4:
        total, period, box, steps, its = 100000, 10, (289.0,) * 3, 10, 10
        types = [rbc_cell_type(3), platelet_cell_type(2)]
        sigma, gamma = 0.2, 0.02
    elif index == 5:
        total, period, box, steps, its = 10000, 0, (139.0,) * 3, 10, 10
        types = [rbc_cell_type(level if level is not None else 4)]
    else:
        total, period, box, steps, its = 114, 6, (50.0, 50.0, 10.0), 20, 5
        types = [rbc_cell_type(3, base="octa"), platelet_cell_type(2, base="octa")]
        sigma, gamma, redraw, dt = 0.2, 0.02, True, 0.25
    if n_cells is not None:
        total = int(n_cells)
    type_of_cell = np.zeros(total, dtype=np.int32)
    if period:
        type_of_cell[period - 1::period] = 1           # every `period`-th cell is a platelet

    positions, velocities, heights = [], [], []
    rot_children = s_rot.spawn(len(types))
    trans_children = s_trans.spawn(len(types))
    for t, ct in enumerate(types):
        count = int(np.sum(type_of_cell == t))
        if index == 1:
            pos = np.broadcast_to(ct.rest_positions, (count,) + ct.rest_positions.shape).copy()
        else:
            rot = _haar_rotations(np.random.Generator(np.random.PCG64(rot_children[t])), count)
            trans = np.random.Generator(np.random.PCG64(trans_children[t])).uniform(
                0.0, 1.0, (count, 3)) * np.asarray(box)
            pos = np.einsum("cij,vj->cvi", rot, ct.rest_positions) + trans[:, None, :]
        positions.append(np.ascontiguousarray(pos))
        velocities.append(np.zeros_like(pos))
        heights.append(pos[..., 2] - 0.5 * box[2])
    return Population(
        name=CONFIG_NAMES[index], types=types, type_of_cell=type_of_cell,
        positions=positions, velocities=velocities, dt=dt, n_steps=steps, n_iterations=its,
        box=box, force_sigma=sigma, shear_gamma=gamma, redraw_noise_each_step=redraw,
        _force_seed=s_force, _shear_height=heights)
