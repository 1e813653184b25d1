"""fp32 EMULATION of the oracle's own arithmetic: the attainable fp32 floor of a parity case.

TEST INFRASTRUCTURE ONLY (never imported by the product).  It is not a second oracle and pins
nothing: it answers "how far from the fp64 oracle does the SAME algorithm land when its state and its
per-element arithmetic are float32", so that the fp32 parity bounds of tests/test_parity_gpu.py can be
stated as a multiple of something measured instead of a guess.

What is float32 here, mirroring what every fp32 CUDA path of this repository stores in float32:
the state x_n, v, F, b, d, g in CELL-LOCAL coordinates (the cell's vertex centroid is subtracted in fp64
first), the displacement form d = x - x_n, and every per-element energy gradient
(the oracle's numpy code, `oracle.npfem_oracle.grad_energy`, called on float32 arrays with a float32
copy of the rest data - numpy keeps float32 throughout).  `two_float=True` (what the library stores since
round 2) keeps the position as an unevaluated float32 pair x + xl and adds d to it with a compensated
sum; `two_float=False` is the plain x <- fl(x + d) of round 1, whose rounding (half an ulp of a ~4 um
coordinate per step against a ~1e-4 um step) turned out to BE the fp32 floor.  What stays fp64: the PBD damping moments
(the CUDA prologue reduces them in fp64) and the H~^-1 solve (the operator is inverted in fp64; only
its operands are rounded).  `tf32=True` additionally rounds g and the increment's operator input to
TF32 (10-bit mantissa, to nearest), the rounding the tensor-core global step adds.
"""
from __future__ import annotations

import dataclasses

import numpy as np

from oracle import npfem_oracle as orc

F32 = np.float32


def _td32(td: orc.TypeData) -> orc.TypeData:
    """The rest data with every per-element float array cast to float32 (indices and the fp64
    matrices untouched)."""
    cast = {}
    for f in ("dm_a", "dm_b", "dm_c", "area0", "theta0", "area_vertex", "mass"):
        cast[f] = getattr(td, f).astype(F32)
    return dataclasses.replace(td, **cast)


def tf32_round(a: np.ndarray) -> np.ndarray:
    """float32 -> nearest value with a 10-bit mantissa (ties away from zero, like cvt.rna.tf32.f32)."""
    u = np.ascontiguousarray(a, dtype=F32).view(np.uint32)
    u = (u + np.uint32(0x1000)) & np.uint32(0xFFFFE000)
    return u.view(F32)


def step_fp32(x_local: np.ndarray, x_low: np.ndarray, v: np.ndarray, f_ext: np.ndarray, td: orc.TypeData,
              td32: orc.TypeData, n_iterations: int, tf32: bool = False, two_float: bool = True):
    """One time step on float32 state in cell-local coordinates; returns (x_local, x_low, v) float32."""
    h = td.h
    v64 = orc.pbd_damping(x_local.astype(np.float64), v.astype(np.float64), td.mass, td.kappa)
    v32 = v64.astype(F32)
    b = (td32.mass[:, None] * v32 / F32(h) + f_ext).astype(F32)
    d = (F32(h) * v32).astype(F32)
    inv_h2 = F32(1.0 / h ** 2)
    m_tilde32 = td.M_tilde.astype(F32)
    for _ in range(n_iterations):
        x = (x_local + (x_low + d).astype(F32)).astype(F32)                   # the rounding every fp32 path makes
        ge = orc.grad_energy(x, td32)
        assert ge.dtype == F32
        md = np.einsum("ij,...jc->...ic", m_tilde32, d).astype(F32)
        g = (md * inv_h2 - b + ge).astype(F32)
        if tf32:
            g = tf32_round(g)
        inc = orc.solve_H_tilde(g.astype(np.float64), td)
        d = (d - inc.astype(F32)).astype(F32)
    t = (x_low + d).astype(F32)
    x_new = (x_local + t).astype(F32)
    x_low = (t - (x_new - x_local).astype(F32)).astype(F32) if two_float else np.zeros_like(x_new)
    return x_new, x_low, (d / F32(h)).astype(F32)


def run_fp32(x0: np.ndarray, v0: np.ndarray, forces_of_step, td: orc.TypeData, n_steps: int, n_iterations: int,
             tf32: bool = False, two_float: bool = True):
    """n_steps steps; x0 [cells, n, 3] fp64 global positions.  Returns fp64 global positions and velocities
    (origin + float32 local state), like get_state(dtype=fp64) of the library."""
    td32 = _td32(td)
    origin = x0.mean(axis=-2, keepdims=True)
    local = x0 - origin
    x = local.astype(F32)
    xl = (local - x.astype(np.float64)).astype(F32) if two_float else np.zeros_like(x)
    v = v0.astype(F32)
    for s in range(n_steps):
        x, xl, v = step_fp32(x, xl, v, forces_of_step(s).astype(F32), td, td32, n_iterations, tf32, two_float)
    return origin + (x.astype(np.float64) + xl.astype(np.float64)), v.astype(np.float64)


def floor_of(pop, n_steps=None, n_iterations=None, tf32: bool = False, two_float: bool = True):
    """Per type (x, v) of the float32 emulation for a workloads.Population (same shape as run_oracle)."""
    n_steps = pop.n_steps if n_steps is None else n_steps
    n_iterations = pop.n_iterations if n_iterations is None else n_iterations
    out = []
    for t, ct in enumerate(pop.types):
        if pop.positions[t].shape[0] == 0:
            out.append((pop.positions[t].copy(), pop.velocities[t].copy()))
            continue
        td = orc.make_type(ct, pop.dt)
        out.append(run_fp32(pop.positions[t], pop.velocities[t], lambda s, t=t: pop.forces(s)[t], td,
                            n_steps, n_iterations, tf32, two_float))
    return out
