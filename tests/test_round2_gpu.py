"""GPU tests added in round 2: the boundary's memory contract (no library-side allocation with caller-owned
workspace + scratch), the collision term under re-centring, the material branches nobody ran
(rayleigh_alpha != 0, rayleigh_beta = 0, kappa_damping = 0), and parity at the sizes BASELINE.json states
(configs[1] at its full 1,000 cells x 10 x 10; configs[3] at 100,000 cells for all 10 steps on sampled cells)."""
import ctypes as C
import dataclasses

import numpy as np
import pytest

from parity_utils import compare, displacement_errors, rel_l2, run_gpu, run_oracle, run_oracle_parallel
from workloads import make_config

pytestmark = pytest.mark.gpu


# ---- boundary: every byte of device memory comes from the caller (north_star: "PyTorch used only for device
# memory and streams"; include/npfem.h npfem_bind_workspace / npfem_bind_scratch) -------------------------------
def test_caller_owned_workspace_and_scratch_no_library_allocations():
    """Raw C ABI through ctypes: create -> workspace_bytes -> bind_workspace -> scratch_bytes -> bind_scratch, then
    diagnostics + line search + collisions + steps.  cudaMemGetInfo (through torch.cuda.mem_get_info) before and
    after: the library itself allocated nothing - not at create (the H~ inverse runs inside the workspace), not
    when the features were switched on, not in npfem_step."""
    import torch
    from paper_1911_03062_b200 import binding
    lib = binding.load_library()
    pop = make_config(3, n_cells=24)
    torch.cuda.init()
    stream = torch.cuda.current_stream(0)
    torch.zeros(1, device="cuda:0")                          # context + allocator warm
    keep, arr = [], (binding._CellType * len(pop.types))()
    for i, ct in enumerate(pop.types):
        rest = np.ascontiguousarray(ct.rest_positions, dtype=np.float64)
        tri = np.ascontiguousarray(ct.triangles, dtype=np.int32)
        keep += [rest, tri]
        arr[i] = binding._CellType(rest.shape[0], tri.shape[0], rest.ctypes.data_as(C.POINTER(C.c_double)),
                                   tri.ctypes.data_as(C.POINTER(C.c_int32)), binding._material_struct(ct.material))
    toc = np.ascontiguousarray(pop.type_of_cell, dtype=np.int32)
    # a throw-away pass through the same calls first: the CUDA runtime loads its modules (and reserves their local
    # memory) at the first launch of each kernel, which is not the library allocating
    warm = binding.Solver(pop.types, pop.type_of_cell, pop.dt, precision="fp32")
    warm.set_option(binding.OPT_DIAGNOSTICS, 1)
    warm.set_line_search(3)
    warm.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
    warm.set_collisions(torch.from_numpy(pop.packed(pop.positions)).cuda(),
                        torch.ones(sum(p.shape[0] * p.shape[1] for p in pop.positions), dtype=torch.float64, device="cuda:0"))
    warm.set_forces(torch.from_numpy(pop.packed(pop.forces(0), dtype=np.float32)).cuda())
    warm.step(6)
    warm.get_objective()
    warm.get_state()
    warm.close()
    del warm
    ctx = C.c_void_p()
    assert lib.npfem_create(C.byref(ctx), arr, len(pop.types), toc.ctypes.data_as(C.POINTER(C.c_int32)), pop.n_cells,
                            pop.dt, binding.NPFEM_F32, 0, C.c_void_p(stream.cuda_stream)) == 0
    features = binding.FEATURE_DIAGNOSTICS | binding.FEATURE_LINE_SEARCH | binding.FEATURE_COLLISIONS
    ws_bytes, sc_bytes = lib.npfem_workspace_bytes(ctx), lib.npfem_scratch_bytes(ctx, features)
    assert sc_bytes > 0 and lib.npfem_scratch_bytes(ctx, 0) == 0
    # enabling a feature on a caller-owned workspace before its scratch is bound is refused, not malloc'ed
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device="cuda:0")
    sc = torch.empty(sc_bytes, dtype=torch.uint8, device="cuda:0")
    x0 = torch.from_numpy(pop.packed(pop.positions)).cuda()
    f0 = torch.from_numpy(pop.packed(pop.forces(0), dtype=np.float32)).cuda()
    tg = torch.from_numpy(pop.packed([p + 0.01 for p in pop.positions])).cuda()
    kk = torch.full((x0.numel() // 3,), 50.0, dtype=torch.float64, device="cuda:0")
    x_out, v_out = torch.empty_like(x0), torch.empty_like(x0)
    hist = torch.empty((7, pop.n_cells), dtype=torch.float64, device="cuda:0")
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info(0)
    assert lib.npfem_bind_workspace(ctx, C.c_void_p(ws.data_ptr()), ws.numel()) == 0
    assert lib.npfem_set_line_search(ctx, 3, 1e-4, 0.0) == -4          # NPFEM_ENOMEM: scratch not bound yet
    assert b"scratch" in lib.npfem_last_error(ctx)
    assert lib.npfem_bind_scratch(ctx, C.c_void_p(sc.data_ptr()), sc.numel() - 256, features) == -4
    assert lib.npfem_bind_scratch(ctx, C.c_void_p(sc.data_ptr()), sc.numel(), features) == 0
    assert lib.npfem_bind_scratch(ctx, C.c_void_p(sc.data_ptr()), sc.numel(), features) == -5   # already bound
    assert lib.npfem_set_option(ctx, binding.OPT_DIAGNOSTICS, 1) == 0
    assert lib.npfem_set_line_search(ctx, 3, 1e-4, 0.0) == 0
    assert lib.npfem_set_state(ctx, None, 0, C.c_void_p(x0.data_ptr()), None, binding.NPFEM_F64, binding.NPFEM_DEVICE) == 0
    assert lib.npfem_set_collisions(ctx, None, 0, C.c_void_p(tg.data_ptr()), C.c_void_p(kk.data_ptr()), binding.NPFEM_F64,
                                    binding.NPFEM_DEVICE) == 0
    assert lib.npfem_set_forces(ctx, None, 0, C.c_void_p(f0.data_ptr()), binding.NPFEM_F32, binding.NPFEM_DEVICE) == 0
    for _ in range(3):
        assert lib.npfem_step(ctx, 6) == 0, lib.npfem_last_error(ctx)
    n_entries = C.c_int32(0)
    assert lib.npfem_get_objective(ctx, C.c_void_p(hist.data_ptr()), 7, C.byref(n_entries), None, binding.NPFEM_DEVICE) == 0
    assert lib.npfem_get_state(ctx, None, 0, C.c_void_p(x_out.data_ptr()), C.c_void_p(v_out.data_ptr()), binding.NPFEM_F64,
                               binding.NPFEM_DEVICE) == 0
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info(0)
    assert free_after == free_before, (free_before, free_after)       # the library took nothing from the device
    assert n_entries.value == 7 and torch.isfinite(hist).all() and torch.isfinite(x_out).all()
    assert (x_out - x0).abs().max() > 0
    # duplicate ids are refused (they would overrun the staging buffers)
    ids = np.array([3, 5, 3], dtype=np.int64)
    assert lib.npfem_get_state(ctx, ids.ctypes.data_as(C.POINTER(C.c_int64)), 3, C.c_void_p(x_out.data_ptr()), None,
                               binding.NPFEM_F64, binding.NPFEM_DEVICE) == -1
    assert b"twice" in lib.npfem_last_error(ctx)
    lib.npfem_destroy(ctx)


def test_default_fp32_path_runs_the_tensor_core_gemm_not_the_simt_fallback():
    """NPFEM_KIND_GLOBAL counts tcgen05 launches only; the SIMT GEMM has its own kind.  On the default fp32 path of
    BASELINE's cell types the SIMT kind must stay at zero (bench.py checks the same on the timed run)."""
    import torch
    from paper_1911_03062_b200 import Solver, binding
    pop = make_config(3, n_cells=330)                         # above the whole-step kernel's batch size for both types
    for math, expect_simt in ((0, False), (1, True)):
        s = Solver(pop.types, pop.type_of_cell, pop.dt, precision="fp32")
        s.set_option(binding.OPT_KERNEL_TIMING, 1)
        s.set_option(binding.OPT_FUSED_STEP, 1)
        s.set_option(binding.OPT_GLOBAL_STEP_MATH, math)
        s.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
        s.set_forces(torch.from_numpy(pop.packed(pop.forces(0))).cuda())
        s.step(4)
        t = s.get_kernel_times()
        s.close()
        tc = sum(n for _, n in t["global"])
        simt = sum(n for _, n in t["global_simt"])
        assert (simt > 0) == expect_simt and (tc > 0) == (not expect_simt), t


# ---- ADVICE (high): collision targets must survive a re-centre of the cell-local frame --------------------------
@pytest.mark.parametrize("precision", ["fp32", "fp64"])
def test_persistent_collisions_on_drifting_cells(precision):
    """A steady 20 pN push per vertex moves every cell by > 2 um in 60 steps: the prologue re-centres the local frame
    several times (threshold 0.5 um).  Collision targets are set ONCE, persist, and travel with nothing: they are
    global coordinates.  Round 1 stored them relative to the origin at call time, so every re-centre added a
    spurious force k * shift to every flagged vertex; this test fails on that build."""
    import torch
    from oracle import npfem_oracle as orc
    from paper_1911_03062_b200 import Solver, binding
    pop = make_config(3, n_cells=12)
    n_steps, n_iterations = 60, 3
    forces = [f.copy() for f in pop.forces(0)]
    for f in forces:
        f[..., 0] += 20.0
    rng = np.random.default_rng(77)
    targets, stiff = [], []
    for t in range(len(pop.types)):
        shape = pop.positions[t].shape[:2]
        stiff.append(np.where(rng.random(shape) < 0.1, rng.uniform(5, 40, shape), 0.0))
        targets.append(pop.positions[t] + np.array([1.0, 0.0, 0.0]) + 0.02 * rng.standard_normal(pop.positions[t].shape))
    np_io = np.float32 if precision == "fp32" else np.float64
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision=precision)
    solver.set_option(binding.OPT_FUSED_STEP, 1)
    solver.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
    solver.set_collisions(torch.from_numpy(pop.packed(targets)).cuda(),
                          torch.from_numpy(pop.packed([k[..., None].repeat(3, -1) for k in stiff])[::3].copy()).cuda())
    solver.set_forces(torch.from_numpy(pop.packed(forces, dtype=np_io)).cuda())
    for _ in range(n_steps):
        solver.step(n_iterations)
    x, v = solver.get_state()
    xs = pop.unpack(x.cpu().numpy())
    solver.close()
    for t, ct in enumerate(pop.types):
        td = orc.make_type(ct, pop.dt)
        xr, _ = orc.run(pop.positions[t], pop.velocities[t], lambda s, t=t: forces[t], td, n_steps, n_iterations,
                        collisions=(targets[t], stiff[t]))
        x_free, _ = orc.run(pop.positions[t], pop.velocities[t], lambda s, t=t: forces[t], td, n_steps, n_iterations)
        x0 = pop.positions[t]
        moved = np.linalg.norm((xr - x0).mean(axis=1), axis=1).min()
        err = displacement_errors(xs[t], xr, x0)
        print(precision, ct.name, err, "moved um", moved, "contacts matter", rel_l2(xr - x0, x_free - x0))
        assert moved > 1.0                                         # several re-centres happened
        assert rel_l2(xr - x0, x_free - x0) > 0.02                 # and the contacts matter
        assert err["disp"] <= (1e-9 if precision == "fp64" else 1e-4), err
        assert err["worst_cell"] <= (1e-9 if precision == "fp64" else 2e-4), err


# ---- VERDICT missing #5: material branches no test ran ------------------------------------------------------------
@pytest.mark.parametrize("alpha,beta,kappa", [(0.3, 0.01, 0.5), (0.0, 0.0, 0.0), (0.0, 0.01, 0.0)])
@pytest.mark.parametrize("precision,config,fused", [("fp64", 3, 1), ("fp32", 3, 1), ("fp32", 6, 2)])
def test_material_branches_alpha_beta_kappa(precision, config, fused, alpha, beta, kappa):
    """rayleigh_alpha != 0 (C = alpha M + beta L: inertia_coef = (1 + h alpha)/h^2 in every kernel),
    rayleigh_beta = 0 (gamma = 0 in the reduced-gradient kernels, no stencil in the generic one) and
    kappa_damping = 0 ("0 = off": the prologue skips the angular moments).  Mixed cell types through the batched
    kernels (config 3: scheduled local step + tcgen05 GEMM in fp32) and through the whole-step kernel (config 6, the
    paper's meshes), a non-zero initial velocity so that the damping terms act.  fp32 bounds: 2 x the values measured
    on B200; with the FP32-FFMA global step the same runs sit on the fp32 floor, so what is left
    with the tensor cores is the TF32 rounding of H~^-1 (largest for the stiff platelets at kappa = 0)."""
    from paper_1911_03062_b200 import binding
    pop = make_config(config, n_cells=34)
    pop.types = [dataclasses.replace(ct, material=dataclasses.replace(ct.material, rayleigh_alpha=alpha, rayleigh_beta=beta,
                                                                      kappa_damping=kappa)) for ct in pop.types]
    rng = np.random.default_rng(5)
    pop.velocities = [2e-3 * rng.standard_normal(p.shape) for p in pop.positions]
    ref = run_oracle(pop, 3, 5)
    variants = [("default", [])] if precision == "fp64" or fused == 2 else [("tf32", []), ("ffma", [(binding.OPT_GLOBAL_STEP_MATH, 1)])]
    for name, options in variants:
        gpu, solver = run_gpu(pop, precision, n_steps=3, n_iterations=5, fused_step=fused, options=options)
        solver.close()
        for r in compare(pop, gpu, ref):
            print(precision, config, name, (alpha, beta, kappa), r)
            if precision == "fp64":
                assert r["pos"] <= 1e-10 and r["disp"] <= 1e-8 and r["vel"] <= 1e-8, r
            elif name == "tf32":
                assert r["pos"] <= 1e-4 and r["disp"] <= 9e-4 and r["worst_cell"] <= 1e-3 and r["vel"] <= 7e-4, r
            else:
                assert r["pos"] <= 1e-4 and r["disp"] <= 2e-4 and r["worst_cell"] <= 5e-4 and r["vel"] <= 3e-4, r


# ---- VERDICT missing #2: parity at the sizes BASELINE.json states ---------------------------------------------------
def test_config2_full_1000_cells_10x10_all_cells():
    """BASELINE configs[1] as stated: 1,000 RBC-642, 10 steps x 10 iterations, fp32 GPU vs fp64 oracle over ALL
    cells ("Oracle parity on configs 1-3 over all cells").  The oracle runs cell chunks in a process
    pool (cells are independent; the oracle itself is untouched)."""
    pop = make_config(2)
    assert pop.n_cells == 1000 and pop.n_steps == 10 and pop.n_iterations == 10
    gpu, solver = run_gpu(pop, "fp32")
    solver.close()
    ref = run_oracle_parallel(pop)
    (r,) = compare(pop, gpu, ref)
    print("config 2, 1000 cells, 10 x 10:", r)
    assert r["pos"] <= 1e-4 and r["worst_cell_pos"] <= 1e-4                    # BASELINE.json's bar
    # measured on B200: disp 1.0e-4 (the TF32 rounding of H~^-1; 1.8e-5 with the FP32 or split-operator GEMM, fp32 floor
    # of the two-float state 2.2e-5, of a plain fp32 state 1.8e-4: DESIGN.md section 5)
    assert r["disp"] <= 2e-4 and r["worst_cell"] <= 2.5e-4 and r["worst_vertex"] <= 1.5e-3 and r["vel"] <= 3e-4, r


def test_config4_full_size_all_10_steps_sampled_cells():
    """BASELINE configs[3] exactly as stated and as bench.py times it: 100,000 mixed cells, fp32, default kernels,
    ALL 10 steps x 10 iterations; the oracle recomputes 200 seeded cells per type one by one (first and last slot
    included) - "after 10 steps ... at 100k mixed cells" of the north star."""
    import torch
    from paper_1911_03062_b200 import Solver
    pop = make_config(4)
    assert pop.n_cells == 100000 and pop.n_steps == 10 and pop.n_iterations == 10
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision="fp32")
    solver.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
    solver.set_forces(torch.from_numpy(pop.packed(pop.forces(0), dtype=np.float32)).cuda())
    for _ in range(pop.n_steps):
        solver.step(pop.n_iterations)
    rng = np.random.default_rng(404)
    picked = []
    for t in range(len(pop.types)):
        ids = pop.cells_of_type(t)
        picked.append(ids[np.unique(np.concatenate(([0, ids.size - 1], rng.integers(0, ids.size, 200))))])
    ids = np.sort(np.concatenate(picked))
    x, v = solver.get_state(cell_ids=ids)
    solver.close()
    sub = pop.subset(ids)
    gpu = list(zip(sub.unpack(x.cpu().numpy()), sub.unpack(v.cpu().numpy())))
    ref = run_oracle_parallel(sub, pop.n_steps, pop.n_iterations)
    for r in compare(sub, gpu, ref):
        print("config 4 full size, 10 x 10:", r)
        assert r["pos"] <= 1e-4 and r["worst_cell_pos"] <= 1e-4
        assert r["disp"] <= 1e-4 and r["worst_cell"] <= 1e-3 and r["vel"] <= 3e-4, r


def test_step_is_capturable_in_a_cuda_graph_and_replays_bit_identically():
    """npfem_step allocates nothing and never synchronises (the memory contract of include/npfem.h), so a whole time
    step - prologue, K x (local step, tensor-core global step), epilogue - is ONE capturable launch sequence: captured
    once, replayed, the state equals the eagerly stepped one bit for bit (bench.py --graph times the replays)."""
    import torch
    from paper_1911_03062_b200 import Solver
    pop = make_config(3, n_cells=330)
    side = torch.cuda.Stream()
    x0 = torch.from_numpy(pop.packed(pop.positions)).cuda()
    f0 = torch.from_numpy(pop.packed(pop.forces(0), dtype=np.float32)).cuda()
    torch.cuda.synchronize()
    states = {}
    with torch.cuda.stream(side):
        for mode in ("eager", "graph"):
            solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision="fp32")
            solver.set_state(x0)
            solver.set_forces(f0)
            solver.step(5)                                     # first step eagerly in both runs: attributes, module loads
            if mode == "eager":
                for _ in range(3):
                    solver.step(5)
            else:
                side.synchronize()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=side):
                    solver.step(5)                             # captured, not run
                for _ in range(3):
                    g.replay()
            x, v = solver.get_state()
            side.synchronize()
            states[mode] = (x.cpu().numpy(), v.cpu().numpy())
            solver.close()
    assert np.array_equal(states["eager"][0], states["graph"][0]) and np.array_equal(states["eager"][1], states["graph"][1])
    assert np.abs(states["graph"][0] - pop.packed(pop.positions)).max() > 0
