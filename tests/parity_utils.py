"""Shared helpers of the GPU parity tests: run a workloads.Population through the C-ABI binding
and through the fp64 oracle on the SAME seeded arrays, and compare."""
import numpy as np

from oracle import npfem_oracle as orc


def run_oracle(pop, n_steps=None, n_iterations=None):
    """-> per-type (x, v) after the run, fp64."""
    n_steps = pop.n_steps if n_steps is None else n_steps
    n_iterations = pop.n_iterations if n_iterations is None else n_iterations
    out = []
    for t, ct in enumerate(pop.types):
        if pop.positions[t].shape[0] == 0:
            out.append((pop.positions[t].copy(), pop.velocities[t].copy()))
            continue
        td = orc.make_type(ct, pop.dt)
        out.append(orc.run(pop.positions[t], pop.velocities[t], lambda s, t=t: pop.forces(s)[t], td,
                           n_steps, n_iterations))
    return out


_POOL_POP = None


def _oracle_chunk(job):
    """Worker of run_oracle_parallel (forked: inherits the population through _POOL_POP; numpy only, no CUDA)."""
    t, lo, hi, n_steps, n_iterations = job
    try:
        import threadpoolctl
        threadpoolctl.threadpool_limits(1)
    except Exception:  # pragma: no cover
        pass
    pop = _POOL_POP
    td = orc.make_type(pop.types[t], pop.dt)
    sl = slice(lo, hi)
    return t, lo, orc.run(pop.positions[t][sl], pop.velocities[t][sl], lambda s: pop.forces(s)[t][sl], td,
                          n_steps, n_iterations)


def run_oracle_parallel(pop, n_steps=None, n_iterations=None, workers=None, chunk=8):
    """run_oracle with the cells spread over a process pool: cells are independent within a step,
    so chunks of a bucket are separate oracle runs.  The oracle is called as it stands; only the batching differs."""
    import multiprocessing as mp
    import os
    global _POOL_POP
    n_steps = pop.n_steps if n_steps is None else n_steps
    n_iterations = pop.n_iterations if n_iterations is None else n_iterations
    workers = workers or max(1, len(os.sched_getaffinity(0)))
    jobs = [(t, lo, min(lo + chunk, pop.positions[t].shape[0]), n_steps, n_iterations)
            for t in range(len(pop.types)) for lo in range(0, pop.positions[t].shape[0], chunk)]
    out = [(pop.positions[t].copy(), pop.velocities[t].copy()) for t in range(len(pop.types))]
    if not pop.redraw_noise_each_step:
        pop.forces(0)                                    # draw the constant forces once, before the fork
    _POOL_POP = pop
    try:
        with mp.get_context("fork").Pool(workers) as pool:
            for t, lo, (x, v) in pool.imap_unordered(_oracle_chunk, jobs):
                out[t][0][lo:lo + x.shape[0]] = x
                out[t][1][lo:lo + v.shape[0]] = v
    finally:
        _POOL_POP = None
    return out


def run_gpu(pop, precision, n_steps=None, n_iterations=None, io="fp64", where="device", options=(), fused_step=1):
    """-> per-type (x, v) after the run as fp64 numpy, plus the solver (still open).
    fused_step: NPFEM_OPT_FUSED_STEP (1 = batched kernels, the path the large workloads take; 2 = the
    whole-step kernel of the small-batch path; 0 = the library's own choice by batch size)."""
    import torch
    from paper_1911_03062_b200 import Solver, binding
    n_steps = pop.n_steps if n_steps is None else n_steps
    n_iterations = pop.n_iterations if n_iterations is None else n_iterations
    np_dt = np.float32 if io == "fp32" else np.float64
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision=precision)
    solver.set_option(binding.OPT_FUSED_STEP, fused_step)
    for opt, val in options:
        solver.set_option(opt, val)

    def to_buf(per_type):
        flat = pop.packed(per_type, dtype=np_dt)
        return torch.from_numpy(flat).cuda() if where == "device" else flat

    solver.set_state(to_buf(pop.positions), to_buf(pop.velocities))
    const_forces = None if pop.redraw_noise_each_step else to_buf(pop.forces(0))
    for s in range(n_steps):
        solver.set_forces(const_forces if const_forces is not None else to_buf(pop.forces(s)))
        solver.step(n_iterations)
    x, v = solver.get_state(dtype=io, where=where)
    if where == "device":
        x, v = x.cpu().numpy(), v.cpu().numpy()
    xs, vs = pop.unpack(x.astype(np.float64)), pop.unpack(v.astype(np.float64))
    return list(zip(xs, vs)), solver


def rel_l2(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def displacement_errors(xg, xr, x0):
    """Displacement-relative errors of one type, [cells, n, 3] arrays:
    disp        relative L2 over all cells (the aggregate SURVEY.md R16 asks to report),
    worst_cell  max over cells of the cell's own relative L2 (a bug confined to few cells shows here),
    worst_vertex max over vertices of |error| / (RMS vertex displacement of that cell): a localised error
                (e.g. the two overflow vertices of RBC-642 on 640 threads) cannot hide behind the 642-vertex sum."""
    dg, dr = xg - x0, xr - x0
    err = np.linalg.norm(dg - dr, axis=-1)                                  # [cells, n]
    cell_norm = np.linalg.norm(dr.reshape(dr.shape[0], -1), axis=1)
    rms = cell_norm / np.sqrt(dr.shape[1])
    return {
        "disp": rel_l2(dg, dr),
        "worst_cell": float(np.max(np.linalg.norm(err, axis=1) / cell_norm)),
        "worst_vertex": float(np.max(err / rms[:, None])),
    }


def compare(pop, gpu, ref):
    """Per type: relative L2 error on positions (BASELINE.json's bar), on the displacement
    x_end - x_0 (sharper: aggregate, worst cell, worst vertex) and on velocities."""
    rows = []
    for t in range(len(pop.types)):
        if pop.positions[t].shape[0] == 0:
            continue
        xg, vg = gpu[t]
        xr, vr = ref[t]
        x0 = pop.positions[t]
        row = {
            "type": pop.types[t].name,
            "pos": rel_l2(xg, xr),
            "vel": rel_l2(vg, vr),
            "worst_cell_pos": float(np.max(np.linalg.norm((xg - xr).reshape(xg.shape[0], -1), axis=1)
                                           / np.linalg.norm(xr.reshape(xr.shape[0], -1), axis=1))),
        }
        row.update(displacement_errors(xg, xr, x0))
        rows.append(row)
    return rows
