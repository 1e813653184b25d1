"""Static multi-GPU partition of the cell population.

"Blood cells are distributed evenly and statically to the available GPUs": cells are
independent within a solver step, so the path shards by cell with NO collective inside
the solver.  Each rank owns, per cell type, one contiguous range of that type's cells (in cell-id
order), builds its own `Solver` on them (H~^-1 replicated per GPU) and steps alone; the only exchange
is forces in / state out, done here on the host side of the boundary with `torch.distributed`.

Buffers follow the binding's convention: flat, the listed cells back to back, each `[n(type)][3]`.
"""
from __future__ import annotations

import numpy as np


def static_partition(type_of_cell, world_size: int) -> list[np.ndarray]:
    """Global cell ids owned by each rank (ascending).

    Per type the cells are cut into `world_size` contiguous ranges whose sizes differ by at most one;
    the ranks that get the extra cell rotate from type to type so that the totals stay balanced too.
    """
    if world_size < 1:
        raise ValueError("world_size must be >= 1")
    toc = np.asarray(type_of_cell, dtype=np.int64)
    owned: list[list[np.ndarray]] = [[] for _ in range(world_size)]
    first_extra = 0
    for t in np.unique(toc):
        ids = np.flatnonzero(toc == t)
        base, extra = divmod(ids.shape[0], world_size)
        start = 0
        for k in range(world_size):
            rank = (first_extra + k) % world_size
            size = base + (1 if k < extra else 0)
            owned[rank].append(ids[start:start + size])
            start += size
        first_extra = (first_extra + extra) % world_size
    return [np.sort(np.concatenate(o)) if o else np.zeros(0, dtype=np.int64) for o in owned]


class Partition:
    """Index bookkeeping between the global flat buffers and one rank's flat buffers."""

    def __init__(self, type_of_cell, n_vertices_of_type, world_size: int):
        self.type_of_cell = np.asarray(type_of_cell, dtype=np.int32)
        self.world_size = int(world_size)
        nv = np.asarray(n_vertices_of_type, dtype=np.int64)[self.type_of_cell]
        self.cell_len = 3 * nv                                        # scalars per cell in a flat buffer
        self.cell_off = np.concatenate([[0], np.cumsum(self.cell_len)])  # [n_cells + 1]
        self.cell_ids = static_partition(self.type_of_cell, self.world_size)
        self.counts = [int(self.cell_len[ids].sum()) for ids in self.cell_ids]

    def flat_index(self, rank: int) -> np.ndarray:
        """Positions, in the global flat buffer, of rank's flat buffer entries (in its own order)."""
        ids = self.cell_ids[rank]
        if ids.shape[0] == 0:
            return np.zeros(0, dtype=np.int64)
        lens = self.cell_len[ids]
        starts = np.repeat(self.cell_off[ids], lens)
        within = np.arange(int(lens.sum()), dtype=np.int64) - np.repeat(np.cumsum(lens) - lens, lens)
        return starts + within

    def scatter(self, global_flat, rank: int):
        """Rank's part of a global flat buffer (numpy array or torch tensor)."""
        idx = self.flat_index(rank)
        if isinstance(global_flat, np.ndarray):
            return np.ascontiguousarray(global_flat.reshape(-1)[idx])
        import torch
        return global_flat.reshape(-1)[torch.as_tensor(idx, device=global_flat.device)].contiguous()

    def assemble(self, parts, out=None):
        """Global flat numpy buffer from the per-rank flat buffers."""
        parts = [np.asarray(p).reshape(-1) for p in parts]
        if out is None:
            out = np.empty(int(self.cell_off[-1]), dtype=parts[0].dtype)
        for rank, p in enumerate(parts):
            out[self.flat_index(rank)] = p
        return out


class ShardedSolver:
    """One rank's shard of a statically partitioned population.

    `solver_factory(cell_types, type_of_cell_local, dt, **kw)` defaults to the CUDA `Solver`.  Global
    buffers may be handed to `set_state` / `set_forces` on every rank (each takes its own part);
    `gather_state` returns the global state on every rank (all_gather of host buffers padded to the
    largest shard; no solver kernel waits on another rank).
    """

    def __init__(self, cell_types, type_of_cell, dt: float, rank: int, world_size: int, solver_factory=None, **kw):
        if solver_factory is None:
            from .binding import Solver as solver_factory
        self.rank, self.world_size = int(rank), int(world_size)
        nv = [int(ct.rest_positions.shape[0]) for ct in cell_types]
        self.partition = Partition(type_of_cell, nv, world_size)
        self.cell_ids = self.partition.cell_ids[self.rank]
        self.local_type_of_cell = self.partition.type_of_cell[self.cell_ids]
        self.solver = solver_factory(cell_types, self.local_type_of_cell, dt, **kw)

    def set_state(self, global_positions, global_velocities=None) -> None:
        p = self.partition.scatter(global_positions, self.rank)
        v = None if global_velocities is None else self.partition.scatter(global_velocities, self.rank)
        self.solver.set_state(p, v)

    def set_forces(self, global_forces) -> None:
        self.solver.set_forces(self.partition.scatter(global_forces, self.rank))

    def step(self, n_iterations: int) -> None:
        self.solver.step(n_iterations)

    def local_state(self, dtype="fp64"):
        x, v = self.solver.get_state(dtype=dtype, where="host")
        return np.asarray(x), np.asarray(v)

    def gather_state(self, dtype="fp64", group=None):
        """(positions, velocities) of ALL cells as global flat numpy arrays, on every rank."""
        import torch
        import torch.distributed as dist
        x, v = self.local_state(dtype)
        if self.world_size == 1:
            return self.partition.assemble([x]), self.partition.assemble([v])
        longest = max(self.partition.counts)
        mine = torch.zeros(2, max(longest, 1), dtype=torch.from_numpy(x[:0]).dtype)
        mine[0, :x.shape[0]] = torch.from_numpy(x)
        mine[1, :v.shape[0]] = torch.from_numpy(v)
        parts = [torch.empty_like(mine) for _ in range(self.world_size)]
        dist.all_gather(parts, mine, group=group)
        xs = [parts[r][0, :self.partition.counts[r]].numpy() for r in range(self.world_size)]
        vs = [parts[r][1, :self.partition.counts[r]].numpy() for r in range(self.world_size)]
        return self.partition.assemble(xs), self.partition.assemble(vs)
