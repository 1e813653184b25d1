"""GPU parity: the CUDA path through the C-ABI against the fp64 oracle, element by element on the
same seeded inputs.  Tolerances (BASELINE.json north_star): relative L2 on positions 1e-10 (fp64)
and 1e-4 (fp32).  That bar cannot fail (positions carry the placement offset), so every test also bounds
the DISPLACEMENT error three ways (aggregate, worst cell, worst vertex: parity_utils.displacement_errors)
and the velocity error.  fp64: 1e-8.  fp32: per test, at most 2 x the value measured on B200 and (for the
aggregate) at most 1e-3; the measured values and the emulated fp32 floor they sit on are tabulated in
DESIGN.md section 5."""
import numpy as np
import pytest

from parity_utils import compare, rel_l2, run_gpu, run_oracle
from workloads import icosahedron_cell_type, make_config
from workloads.populations import Population

pytestmark = pytest.mark.gpu

TOL_POS = {"fp64": 1e-10, "fp32": 1e-4}
TOL_FP64 = 1e-8          # displacement / velocity, fp64
# fp32 tests that are not about precision (violent line-search cases, where the cells deform by a good fraction of
# their size and a different backtracking decision moves the result): the bound of the round-1 suite, kept for those
TOL_DISP = {"fp64": TOL_FP64, "fp32": 5e-3}


def assert_row(r, precision, fp32):
    """fp32 = (disp, worst_cell, worst_vertex, vel): <= 2 x the values measured on B200."""
    assert r["pos"] <= TOL_POS[precision] and r["worst_cell_pos"] <= TOL_POS[precision], r
    if precision == "fp64":
        assert r["disp"] <= TOL_FP64 and r["worst_cell"] <= TOL_FP64 and r["worst_vertex"] <= TOL_FP64 and r["vel"] <= TOL_FP64, r
    else:
        disp, worst_cell, worst_vertex, vel = fp32
        assert disp <= 1e-3
        assert r["disp"] <= disp and r["worst_cell"] <= worst_cell and r["worst_vertex"] <= worst_vertex and r["vel"] <= vel, (r, fp32)


def _check(pop, precision, fp32=None, **kw):
    gpu, solver = run_gpu(pop, precision, **kw)
    ref = run_oracle(pop, kw.get("n_steps"), kw.get("n_iterations"))
    rows = compare(pop, gpu, ref)
    solver.close()
    for r in rows:
        print(precision, r)
        assert_row(r, precision, fp32)
    return rows


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_config1_single_rbc(precision):
    # one step from rest: the displacement is ~1e-5 um, its fp32 error is the rounding of x + d itself
    # measured (disp, worst cell, worst vertex, vel): 1.8e-4, 1.8e-4, 5.6e-4, 1.8e-4
    _check(make_config(1), precision, fp32=(3.7e-4, 3.7e-4, 1.2e-3, 3.7e-4))


@pytest.mark.parametrize("precision", ["fp32", "fp64"])
def test_config2_reduced_70_cells_full_schedule(precision):
    # 70 cells = 210 GEMM rows: several 64-row tiles and a ragged tail; full 10 steps x 10 its
    # measured 9.9e-5, 1.1e-4, 6.9e-4, 1.6e-4 (emulated floor of the two-float state 2.2e-5; the rest is the TF32
    # rounding of H~^-1: 2.3e-5 with the split-operator GEMM)
    _check(make_config(2, n_cells=70), precision, fp32=(2e-4, 2.3e-4, 1.4e-3, 3.2e-4))


@pytest.mark.parametrize("precision", ["fp32", "fp64"])
def test_config3_mixed_types_redrawn_forces(precision):
    pop = make_config(3, n_cells=45)          # 41 RBC-642 + 4 PLT-162, interleaved ids
    # measured RBC-642 3.7e-5, 4.0e-4, 1.3e-3, 6.5e-5 (floor 3.1e-5, 4.3e-4, 1.5e-3, 6.1e-5: one cell that hardly moves),
    # PLT-162 1.4e-5, 1.5e-5, 4.4e-5, 1.6e-5
    _check(pop, precision, fp32=(8e-5, 8e-4, 2.7e-3, 1.4e-4), n_steps=4, n_iterations=5)


@pytest.mark.parametrize("precision,impl", [("fp32", 0), ("fp32", 1), ("fp32", 4), ("fp32", 6), ("fp64", 0)])
def test_config5_level4_mesh(precision, impl):
    # 2562 vertices / 5120 triangles: too large for one pass of the quad kernel -> multi-pass quad kernel (fp32 default
    # = impl 6: 4 passes of 640 quads), the large-mesh kernel of round 1 (impl 4: corner forces in chunks) or the
    # generic kernel with its global scratch (impl 1, fp64)
    from paper_1911_03062_b200 import binding
    # measured 2.4e-4, 2.6e-4, 1.3e-3, 2.5e-4 (large-mesh kernel), 2.1e-4, 2.2e-4, 9.7e-4, 2.1e-4 (generic)
    _check(make_config(5, n_cells=40), precision, fp32=(5e-4, 5.2e-4, 2.7e-3, 5.1e-4), n_steps=2, n_iterations=3,
           options=[(binding.OPT_LOCAL_STEP_IMPL, impl)])


def test_icosahedron_cell_fp64():
    ct = icosahedron_cell_type(3.0)
    rng = np.random.default_rng(0)
    pos = ct.rest_positions[None] + 0.05 * rng.standard_normal((5, 12, 3)) + rng.uniform(0, 50, (5, 1, 3))
    pop = Population(name="ico", types=[ct], type_of_cell=np.zeros(5, np.int32), positions=[pos],
                     velocities=[0.02 * rng.standard_normal(pos.shape)], dt=0.1, n_steps=3, n_iterations=8,
                     box=(50.0,) * 3, force_sigma=2.0, shear_gamma=0.0, redraw_noise_each_step=False,
                     _force_seed=np.random.SeedSequence(5), _shear_height=[pos[..., 2]])
    _check(pop, "fp64")


def test_io_paths_agree_and_partial_ids():
    """Host and device buffers, fp32 and fp64 I/O, full and partial id lists give the same state."""
    import torch
    from paper_1911_03062_b200 import Solver
    pop = make_config(3, n_cells=23)
    gpu_dev, s1 = run_gpu(pop, "fp32", n_steps=2, n_iterations=3, io="fp64", where="device")
    gpu_host, s2 = run_gpu(pop, "fp32", n_steps=2, n_iterations=3, io="fp64", where="host")
    for (xa, va), (xb, vb) in zip(gpu_dev, gpu_host):
        assert np.array_equal(xa, xb) and np.array_equal(va, vb)
    ids = np.array([21, 3, 10, 0], dtype=np.int64)          # cell 10 and 21 are platelets
    xs, vs = s1.get_state(cell_ids=ids)
    sub = pop.unpack(xs.cpu().numpy(), ids)
    order_rbc = [3, 0]                                       # list order within each type
    assert np.array_equal(sub[0][0], gpu_dev[0][0][3]) and np.array_equal(sub[0][1], gpu_dev[0][0][0])
    assert np.array_equal(sub[1][0], gpu_dev[1][0][1]) and np.array_equal(sub[1][1], gpu_dev[1][0][0])
    # fp32 read-back is the fp64 read-back rounded once
    x32, _ = s1.get_state(dtype="fp32")
    x64, _ = s1.get_state(dtype="fp64")
    assert torch.equal(x32, x64.to(torch.float32))
    s1.close()
    s2.close()


def test_partial_set_state_and_forces_persist():
    from paper_1911_03062_b200 import Solver, NpfemError
    import torch
    pop = make_config(2, n_cells=6)
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision="fp64")
    first, rest = np.array([0, 1, 2]), np.array([5, 4, 3])
    solver.set_state(torch.from_numpy(pop.packed(pop.positions, first)).cuda(), cell_ids=first)
    with pytest.raises(NpfemError) as e:
        solver.step(2)                                        # three cells still have no state
    assert e.value.code == -5
    solver.set_state(torch.from_numpy(pop.packed(pop.positions, rest)).cuda(), cell_ids=rest)
    solver.set_forces(torch.from_numpy(pop.packed(pop.forces(0))).cuda())
    solver.step(4)
    solver.step(4)                                            # forces persist until overwritten
    x, v = solver.get_state()
    ref = run_oracle(pop, 2, 4)
    assert rel_l2(pop.unpack(x.cpu().numpy())[0], ref[0][0]) < 1e-10
    with pytest.raises(NpfemError) as e:
        solver.step(0)
    assert e.value.code == -1
    solver.close()


def test_rest_state_stays_at_rest_far_from_origin():
    """P1 on the GPU: rigidly placed rest shapes, no force -> no motion, even 1000 um out in fp32."""
    from paper_1911_03062_b200 import Solver
    import torch
    pop = make_config(2, n_cells=8)
    pos = [pop.positions[0] + 1000.0]
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision="fp32")
    solver.set_state(torch.from_numpy(pop.packed(pos)).cuda())
    for _ in range(3):
        solver.step(5)
    x, v = solver.get_state()
    disp = x.cpu().numpy() - pop.packed(pos)
    assert np.abs(disp).max() < 2e-6          # fp32 round-off of the local coordinates only
    assert np.abs(v.cpu().numpy()).max() < 1e-4
    solver.close()


def test_zero_cells_and_empty_bucket():
    from paper_1911_03062_b200 import Solver
    pop = make_config(3, n_cells=5)                           # 5 RBCs, platelet bucket empty
    gpu, solver = run_gpu(pop, "fp64", n_steps=1, n_iterations=2)
    ref = run_oracle(pop, 1, 2)
    assert rel_l2(gpu[0][0], ref[0][0]) < 1e-10
    solver.close()
    empty = Solver(pop.types, np.zeros(0, np.int32), pop.dt, precision="fp32")
    empty.step(3)
    x, v = empty.get_state()
    assert x.numel() == 0
    empty.close()


@pytest.mark.parametrize("config", [2, 5])     # 5: RBC-2562, the objective kernel's one-CTA-per-SM variant
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_objective_history_matches_oracle(precision, config):
    from oracle import npfem_oracle as orc
    from paper_1911_03062_b200 import binding
    pop = make_config(config, n_cells=4)
    gpu, solver = run_gpu(pop, precision, n_steps=1, n_iterations=6,
                          options=[(binding.OPT_DIAGNOSTICS, 1)])
    hist, mono = solver.get_objective()
    solver.close()
    td = orc.make_type(pop.types[0], pop.dt)
    _, _, rec = orc.step(pop.positions[0], pop.velocities[0], pop.forces(0)[0], td, 6, record=True)
    ref = np.array(rec["objective"])                          # [7, 4]
    assert hist.shape == ref.shape
    scale = np.abs(ref).max()
    assert np.abs(hist - ref).max() < (1e-9 if precision == "fp64" else 2e-3) * scale
    assert np.all(mono == 1)


def test_tf32_tensor_core_global_step_vs_fp32_ffma():
    """The tcgen05/TF32 global step and the exact FP32-FFMA global step give the same trajectory up
    to TF32 rounding of the (small) increment; both stay within the fp32 bar against the oracle."""
    from paper_1911_03062_b200 import binding
    pop = make_config(3, n_cells=90)                  # 82 RBC (246 rows: 2 M tiles, ragged) + 8 PLT
    tf32, s1 = run_gpu(pop, "fp32", n_steps=3, n_iterations=5, options=[(binding.OPT_GLOBAL_STEP_MATH, 0)])
    ffma, s2 = run_gpu(pop, "fp32", n_steps=3, n_iterations=5, options=[(binding.OPT_GLOBAL_STEP_MATH, 1)])
    s1.close()
    s2.close()
    ref = run_oracle(pop, 3, 5)
    for t in range(2):
        x0 = pop.positions[t]
        d_tf32, d_ffma, d_ref = tf32[t][0] - x0, ffma[t][0] - x0, ref[t][0] - x0
        print(pop.types[t].name, "tf32 vs ffma", rel_l2(d_tf32, d_ffma), "tf32 vs oracle", rel_l2(d_tf32, d_ref),
              "ffma vs oracle", rel_l2(d_ffma, d_ref))
        # measured: tf32 vs ffma 4.0e-5 / 1.7e-5, tf32 vs oracle 5.5e-5 / 1.7e-5, ffma vs oracle 4.9e-5 / 6.7e-6
        assert rel_l2(d_tf32, d_ffma) < 8e-5
        assert rel_l2(tf32[t][0], ref[t][0]) < 1e-4
        assert rel_l2(d_tf32, d_ref) < 1.1e-4 and rel_l2(d_ffma, d_ref) < 1e-4


@pytest.mark.parametrize("impl", [1, 2, 3, 5])
def test_fp32_local_step_implementations(impl):
    """Every fp32 local-step kernel (1 generic, 2 shared-memory tables, 3 scheduled: register-resident
    topology + colour-assigned conflict-free slots, 5 quad: one thread per pair of adjacent triangles, the default
    where the type allows it) against the oracle; RBC-642 exercises the second vertex pass of the scheduled and quad
    kernels (642 vertices on 640 threads)."""
    from paper_1911_03062_b200 import binding
    pop = make_config(3, n_cells=300)         # 273 RBC + 27 PLT: more cells than one wave of CTAs for PLT
    gpu, solver = run_gpu(pop, "fp32", n_steps=3, n_iterations=5, options=[(binding.OPT_LOCAL_STEP_IMPL, impl)])
    solver.close()
    ref = run_oracle(pop, 3, 5)
    for r in compare(pop, gpu, ref):
        print(impl, r)
        # measured (all three kernels within 10 %): RBC-642 6.1e-5, 6.5e-4, 2.1e-3, 8.8e-5; PLT-162 2.1e-5, 1.0e-4, 2.5e-4, 2.8e-5
        assert_row(r, "fp32", (1.3e-4, 1.3e-3, 4.3e-3, 1.8e-4))


def test_two_pass_mesh_with_a_partly_filled_last_pass():
    """An octahedral RBC mesh of 1,026 vertices / 2,048 triangles: 1,024 quads = one full pass of the multi-pass quad
    kernel + one pass of 384 quads (threads without a quad, vertices listed in both passes)."""
    from paper_1911_03062_b200 import binding
    from workloads.meshes import rbc_cell_type
    ct = rbc_cell_type(4, base="octa")
    assert ct.rest_positions.shape[0] == 1026 and binding.quad_schedule_stats(ct, 0.1, multipass=True)["threads"] == 2
    rng = np.random.default_rng(5)
    n_cells = 170                               # more cells than CTAs: the persistent loop wraps
    pos = ct.rest_positions[None] + rng.uniform(0, 120, (n_cells, 1, 3))
    pop = Population(name="octa4", types=[ct], type_of_cell=np.zeros(n_cells, np.int32), positions=[pos],
                     velocities=[0.01 * rng.standard_normal(pos.shape)], dt=0.1, n_steps=2, n_iterations=4,
                     box=(120.0,) * 3, force_sigma=1.0, shear_gamma=0.0, redraw_noise_each_step=False,
                     _force_seed=np.random.SeedSequence(6), _shear_height=[pos[..., 2]])
    ref = run_oracle(pop)
    out = {}
    for impl in (6, 1):
        gpu, solver = run_gpu(pop, "fp32", options=[(binding.OPT_LOCAL_STEP_IMPL, impl), (binding.OPT_GLOBAL_STEP_MATH, 1)])
        solver.close()
        out[impl] = compare(pop, gpu, ref)[0]
        print(impl, out[impl])
    # the generic kernel (impl 1) is the yardstick on the same inputs: the multi-pass kernel sits at the same fp32 floor
    for k in ("disp", "worst_cell", "worst_vertex", "vel"):
        assert out[6][k] <= 1.5 * out[1][k] + 1e-6, (k, out[6][k], out[1][k])
    assert out[6]["pos"] <= TOL_POS["fp32"] and out[6]["disp"] <= 5e-4


def test_multipass_kernel_on_an_irregular_level4_mesh_valence_up_to_8():
    """2,562 vertices after 400 random edge flips (valences 4 .. 8): the 8-read variant of the multi-pass quad kernel
    against the generic kernel on the same inputs and against the oracle."""
    from paper_1911_03062_b200 import binding
    from workloads.meshes import irregular_cell_type
    ct = irregular_cell_type(4, 400, seed=5)
    assert np.bincount(ct.triangles.ravel()).max() == 8
    st = binding.quad_schedule_stats(ct, 0.1, multipass=True)
    assert st["valid"] == 1 and st["threads"] == 4 and st["reads_per_vertex"] == 8 and st["consistent"] == 1
    rng = np.random.default_rng(17)
    n_cells = 12
    pos = ct.rest_positions[None] + rng.uniform(0, 90, (n_cells, 1, 3))
    pop = Population(name="irr4", types=[ct], type_of_cell=np.zeros(n_cells, np.int32), positions=[pos],
                     velocities=[0.01 * rng.standard_normal(pos.shape)], dt=0.1, n_steps=2, n_iterations=3,
                     box=(90.0,) * 3, force_sigma=1.0, shear_gamma=0.0, redraw_noise_each_step=False,
                     _force_seed=np.random.SeedSequence(18), _shear_height=[pos[..., 2]])
    ref = run_oracle(pop)
    out = {}
    for impl in (6, 1):
        gpu, solver = run_gpu(pop, "fp32", options=[(binding.OPT_LOCAL_STEP_IMPL, impl), (binding.OPT_GLOBAL_STEP_MATH, 1)])
        solver.close()
        out[impl] = compare(pop, gpu, ref)[0]
        print(impl, out[impl])
    for k in ("disp", "worst_cell", "worst_vertex", "vel"):
        assert out[6][k] <= 1.5 * out[1][k] + 1e-6, (k, out[6][k], out[1][k])
    assert out[6]["pos"] <= TOL_POS["fp32"] and out[6]["disp"] <= TOL_DISP["fp32"]


@pytest.mark.parametrize("precision,impl", [("fp64", 0), ("fp32", 1), ("fp32", 3), ("fp32", 5)])
def test_irregular_mesh_valence_up_to_8(precision, impl):
    """A mesh that is not an icosphere (flipped edges, valences 4..8): generic kernels and the
    8-read variant of the scheduled kernel against the oracle."""
    from paper_1911_03062_b200 import binding
    from workloads.meshes import irregular_cell_type
    ct = irregular_cell_type(2, 40, seed=3)
    val = np.bincount(ct.triangles.ravel())
    assert val.max() > 6
    rng = np.random.default_rng(11)
    n_cells = 37
    pos = ct.rest_positions[None] + rng.uniform(0, 80, (n_cells, 1, 3))
    pop = Population(name="irr", types=[ct], type_of_cell=np.zeros(n_cells, np.int32), positions=[pos],
                     velocities=[0.01 * rng.standard_normal(pos.shape)], dt=0.1, n_steps=3, n_iterations=6,
                     box=(80.0,) * 3, force_sigma=1.0, shear_gamma=0.0, redraw_noise_each_step=False,
                     _force_seed=np.random.SeedSequence(12), _shear_height=[pos[..., 2]])
    gpu, solver = run_gpu(pop, precision, options=[(binding.OPT_LOCAL_STEP_IMPL, impl)], fused_step=2 if impl == 0 else 1)
    solver.close()
    ref = run_oracle(pop)
    for r in compare(pop, gpu, ref):
        print(precision, impl, r)
        # An irregular mesh with slivers (valence 4..8 after random edge flips): the strain invariants of its thin
        # triangles amplify the fp32 rounding.  measured: generic 1.9e-3, 2.7e-3, 6.6e-3, 1.2e-3; scheduled 1.1e-3,
        # 1.6e-3, 3.8e-3, 6.5e-4 - the one test whose aggregate stays above 1e-3 (bound by hand, not by assert_row)
        assert r["pos"] <= TOL_POS[precision], r
        if precision == "fp64":
            assert r["disp"] <= TOL_FP64 and r["vel"] <= TOL_FP64, r
        else:
            assert r["disp"] <= 3.8e-3 and r["worst_cell"] <= 5.4e-3 and r["worst_vertex"] <= 1.4e-2 and r["vel"] <= 2.4e-3, r


def _ls_population(n_cells, h, force_sigma, seed, level=2):
    """RBC-162 cells at rest shape under N(0, force_sigma) forces: with h = 30 us and 3000 pN the plain
    iteration of Eq. (4) diverges (tests/test_oracle_pins.py), the line search must not."""
    from workloads.meshes import rbc_cell_type
    ct = rbc_cell_type(level)
    rng = np.random.default_rng(seed)
    pos = ct.rest_positions[None] + rng.uniform(0, 60, (n_cells, 1, 3))
    return Population(name="ls", types=[ct], type_of_cell=np.zeros(n_cells, np.int32), positions=[pos],
                      velocities=[np.zeros_like(pos)], dt=h, n_steps=1, n_iterations=15, box=(60.0,) * 3,
                      force_sigma=force_sigma, shear_gamma=0.0, redraw_noise_each_step=False,
                      _force_seed=np.random.SeedSequence(seed + 1), _shear_height=[pos[..., 2]])


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_line_search_violent_case_matches_oracle(precision):
    """Armijo backtracking on the GPU against oracle.step_line_search, on a case
    where the plain iteration blows up.  fp64: same step lengths (the decisions are taken in fp64 on
    both sides); errors within the displacement bounds of DESIGN.md section 5 (1e-8 / 5e-3)."""
    import torch
    from oracle import npfem_oracle as orc
    from paper_1911_03062_b200 import Solver
    pop = _ls_population(9, 30.0, 3000.0, seed=21)
    td = orc.make_type(pop.types[0], pop.dt)
    f = pop.forces(0)[0]
    xr, vr, hist = orc.step_line_search(pop.positions[0], pop.velocities[0], f, td, 15, max_halvings=8, c1=1e-4, record=True)
    assert np.array(hist["alpha"]).min() < 1.0                       # the case does backtrack
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision=precision)
    solver.set_line_search(8, 1e-4, 0.0)
    solver.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
    solver.set_forces(torch.from_numpy(pop.packed(pop.forces(0))).cuda())
    solver.step(15)
    x, v = solver.get_state()
    alpha = solver.get_step_lengths()
    solver.close()
    xg = pop.unpack(x.cpu().numpy())[0]
    x0 = pop.positions[0]
    print(precision, "pos", rel_l2(xg, xr), "disp", rel_l2(xg - x0, xr - x0), "alpha gpu", alpha, "oracle", hist["alpha"][-1])
    assert np.all(np.isfinite(xg))
    # the cells deform by a good fraction of their size here, so the position-relative error IS the
    # displacement-relative one: the displacement bound of DESIGN.md section 5 applies to both
    bound = TOL_FP64 if precision == "fp64" else 4e-4               # fp32 measured 1.1e-4 .. 1.6e-4
    assert rel_l2(xg, xr) <= bound
    assert rel_l2(xg - x0, xr - x0) <= bound
    if precision == "fp64":
        assert np.array_equal(alpha, hist["alpha"][-1])
    else:
        assert np.all(np.isin(alpha, 0.5 ** np.arange(0, 9)))
        # the search must not stall: with a plain TF32 search direction every cell rejected all nine step lengths
        # from iteration 11 on (alpha = 2^-8 everywhere, displacement error 2.7e-3); the 3xTF32 direction tracks the
        # oracle's step lengths (1.6e-4)
        assert np.median(alpha) > 0.5 ** 8
        assert rel_l2(xg - x0, xr - x0) <= 1e-3


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_line_search_large_time_step_rbc642(precision):
    """SURVEY.md 8(f)-1's own case on the BASELINE mesh: h = 10 us (100 x the BASELINE step), N(0, 100 pN) forces,
    RBC-642 (fp32: scheduled local step + damping kernel + 3xTF32 product in three column passes)."""
    import torch
    from oracle import npfem_oracle as orc
    from paper_1911_03062_b200 import Solver
    pop = _ls_population(5, 10.0, 100.0, seed=8, level=3)
    td = orc.make_type(pop.types[0], pop.dt)
    xr, vr, hist = orc.step_line_search(pop.positions[0], pop.velocities[0], pop.forces(0)[0], td, 8, max_halvings=6, c1=1e-4,
                                        record=True)
    assert np.all(np.diff(np.array(hist["objective"]), axis=0) <= 0.0)   # the oracle's objective decreases
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision=precision)
    solver.set_line_search(6, 1e-4, 0.0)
    solver.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
    solver.set_forces(torch.from_numpy(pop.packed(pop.forces(0))).cuda())
    solver.step(8)
    x, v = solver.get_state()
    alpha = solver.get_step_lengths()
    solver.close()
    xg = pop.unpack(x.cpu().numpy())[0]
    x0 = pop.positions[0]
    print(precision, "disp", rel_l2(xg - x0, xr - x0), "alpha gpu", alpha, "oracle", hist["alpha"][-1])
    assert np.all(np.isfinite(xg))
    assert rel_l2(xg - x0, xr - x0) <= (TOL_FP64 if precision == "fp64" else 2e-6)   # fp32 measured 7.6e-7 (full steps throughout)
    if precision == "fp64":
        assert np.array_equal(alpha, hist["alpha"][-1])


def test_line_search_violent_case_rbc642_fp32():
    """The violent case on the BASELINE mesh (RBC-642: scheduled local step, 3xTF32 product in three column passes):
    the search backtracks, does not stall, and the result stays within the fp32 displacement bound of the oracle."""
    import torch
    from oracle import npfem_oracle as orc
    from paper_1911_03062_b200 import Solver
    pop = _ls_population(4, 30.0, 3000.0, seed=33, level=3)
    td = orc.make_type(pop.types[0], pop.dt)
    xr, vr, hist = orc.step_line_search(pop.positions[0], pop.velocities[0], pop.forces(0)[0], td, 12, max_halvings=8, c1=1e-4,
                                        record=True)
    assert np.array(hist["alpha"]).min() < 1.0                       # the case does backtrack
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision="fp32")
    solver.set_line_search(8, 1e-4, 0.0)
    solver.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
    solver.set_forces(torch.from_numpy(pop.packed(pop.forces(0))).cuda())
    solver.step(12)
    x, _ = solver.get_state()
    alpha = solver.get_step_lengths()
    solver.close()
    xg = pop.unpack(x.cpu().numpy())[0]
    x0 = pop.positions[0]
    print("disp", rel_l2(xg - x0, xr - x0), "alpha gpu", alpha, "oracle", hist["alpha"][-1])
    assert np.median(alpha) > 0.5 ** 8
    assert rel_l2(xg - x0, xr - x0) <= TOL_DISP["fp32"]


def test_line_search_fp32_fast_kernels_match_the_generic_full_gradient():
    """fp32 line search: the fast local kernels' reduced gradient + the damping part (launch_damping_grad)
    against the generic kernel's full gradient (OPT_LOCAL_STEP_IMPL = 1) and against the oracle, on the
    violent case (which backtracks) and on mixed RBC-642 / PLT-162 cells."""
    import torch
    from oracle import npfem_oracle as orc
    from paper_1911_03062_b200 import Solver, binding
    pop = _ls_population(9, 30.0, 3000.0, seed=21)
    td = orc.make_type(pop.types[0], pop.dt)
    assert td.beta > 0.0                                             # the damping part is not zero here
    xr, _ = orc.step_line_search(pop.positions[0], pop.velocities[0], pop.forces(0)[0], td, 15, max_halvings=8, c1=1e-4)
    out = {}
    for impl in (0, 1):
        solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision="fp32")
        solver.set_option(binding.OPT_LOCAL_STEP_IMPL, impl)
        solver.set_line_search(8, 1e-4, 0.0)
        solver.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
        solver.set_forces(torch.from_numpy(pop.packed(pop.forces(0))).cuda())
        solver.step(15)
        x, _ = solver.get_state()
        out[impl] = pop.unpack(x.cpu().numpy())[0]
        solver.close()
    x0 = pop.positions[0]
    for impl in (0, 1):
        print("impl", impl, "disp error vs oracle", rel_l2(out[impl] - x0, xr - x0))
        assert rel_l2(out[impl] - x0, xr - x0) <= 3.3e-4           # measured 1.1e-4 .. 1.6e-4 (impl 0), 9.1e-5 (impl 1)
    pop = make_config(3, n_cells=40)
    ref = run_oracle(pop, 2, 5)                                      # full steps descend here: plain oracle
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision="fp32")
    solver.set_line_search(4)
    solver.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
    for s in range(2):
        solver.set_forces(torch.from_numpy(pop.packed(pop.forces(s))).cuda())
        solver.step(5)
    x, _ = solver.get_state()
    assert np.all(solver.get_step_lengths() == 1.0)
    solver.close()
    xs = pop.unpack(x.cpu().numpy())
    for t in range(2):
        assert rel_l2(xs[t], ref[t][0]) <= 1e-4


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_line_search_with_collisions_is_neutral_when_full_steps_descend(precision):
    """Line search + PIK collision term (energy in the objective, gradient added after the local step; in fp32 the
    3xTF32 split then happens just before the GEMMs): on a tame case every full step descends, so the result is the
    oracle's plain run with collisions."""
    import torch
    from oracle import npfem_oracle as orc
    from paper_1911_03062_b200 import Solver
    pop = make_config(3, n_cells=12)
    rng = np.random.default_rng(5)
    targets, stiff = [], []
    for t in range(len(pop.types)):
        shape = pop.positions[t].shape[:2]
        stiff.append(np.where(rng.random(shape) < 0.15, rng.uniform(20, 300, shape), 0.0))
        targets.append(pop.positions[t] + 0.02 * rng.standard_normal(pop.positions[t].shape))
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision=precision)
    solver.set_line_search(4)
    solver.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
    solver.set_collisions(pop.packed(targets).astype(np.float64),
                          pop.packed([k[..., None].repeat(3, -1) for k in stiff])[::3].copy().astype(np.float64))
    np_io = np.float64 if precision == "fp64" else np.float32
    for s in range(2):
        solver.set_forces(torch.from_numpy(pop.packed(pop.forces(s), dtype=np_io)).cuda())
        solver.step(5)
    x, _ = solver.get_state()
    assert np.all(solver.get_step_lengths() == 1.0)
    solver.close()
    xs = pop.unpack(x.cpu().numpy())
    for t, ct in enumerate(pop.types):
        td = orc.make_type(ct, pop.dt)
        xr, _ = orc.run(pop.positions[t], pop.velocities[t], lambda s, t=t: pop.forces(s)[t], td, 2, 5,
                        collisions=(targets[t], stiff[t]))
        x0 = pop.positions[t]
        print(precision, ct.name, rel_l2(xs[t], xr), rel_l2(xs[t] - x0, xr - x0))
        assert rel_l2(xs[t], xr) <= TOL_POS[precision]
        assert rel_l2(xs[t] - x0, xr - x0) <= (TOL_FP64 if precision == "fp64" else 1.2e-4)   # fp32 measured 5.5e-5 / 2.1e-5


def test_line_search_is_neutral_on_a_tame_case_and_freezes_by_tolerance():
    import torch
    from paper_1911_03062_b200 import Solver
    pop = make_config(3, n_cells=30)
    ref = run_oracle(pop, 2, 5)                                      # plain oracle: every full step descends here
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision="fp64")
    solver.set_line_search(6)
    solver.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
    for s in range(2):
        solver.set_forces(torch.from_numpy(pop.packed(pop.forces(s))).cuda())
        solver.step(5)
    x, _ = solver.get_state()
    assert np.all(solver.get_step_lengths() == 1.0)
    xs = pop.unpack(x.cpu().numpy())
    for t in range(2):
        assert rel_l2(xs[t], ref[t][0]) <= 1e-10
    # huge tolerance: nothing moves beyond d0 = h v (v = 0 here): positions stay
    solver.set_line_search(6, 1e-4, 1e12)
    x_before, _ = solver.get_state()
    solver.step(3)
    assert np.all(solver.get_step_lengths() == 0.0)
    x_after, v_after = solver.get_state()
    # d = h v_damped: the cells only coast with their (damped) velocity
    assert torch.allclose(x_after, x_before + pop.dt * v_after, rtol=0, atol=1e-12)
    solver.close()


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_median_filtered_forces_and_velocity_cap(precision):
    """one-ring median filter of F_ext in set_forces and the vertex-velocity
    cap in the epilogue against the oracle; mixed cell types (valence 5 and 6: even and odd
    median counts), forces redrawn every step, the cap set so that it really bites."""
    import torch
    from oracle import npfem_oracle as orc
    from paper_1911_03062_b200 import Solver, binding
    pop = make_config(3, n_cells=34)
    n_steps, n_its, v_max = 3, 5, 2.0e-4
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision=precision)
    solver.set_option(binding.OPT_FORCE_MEDIAN_FILTER, 1)
    solver.set_velocity_cap(v_max)
    solver.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
    for s in range(n_steps):
        solver.set_forces(torch.from_numpy(pop.packed(pop.forces(s))).cuda())
        solver.step(n_its)
    x, v = solver.get_state()
    solver.close()
    xs, vs = pop.unpack(x.cpu().numpy()), pop.unpack(v.cpu().numpy())
    for t, ct in enumerate(pop.types):
        td = orc.make_type(ct, pop.dt)
        xr, vr = orc.run(pop.positions[t], pop.velocities[t], lambda s, t=t: pop.forces(s)[t], td, n_steps, n_its,
                         v_max=v_max, median_filter=True)
        x_plain, v_plain = orc.run(pop.positions[t], pop.velocities[t], lambda s, t=t: pop.forces(s)[t], td, n_steps, n_its)
        x0 = pop.positions[t]
        speed = np.linalg.norm(vr, axis=-1)
        assert np.isclose(speed.max(), v_max) and np.linalg.norm(v_plain, axis=-1).max() > v_max   # the cap bites
        assert rel_l2(xr - x0, x_plain - x0) > 0.05                                              # the filter matters
        print(precision, ct.name, rel_l2(xs[t], xr), rel_l2(xs[t] - x0, xr - x0), rel_l2(vs[t], vr))
        assert rel_l2(xs[t], xr) <= TOL_POS[precision]
        # fp32 measured: disp 7.5e-5 / 2.3e-5, vel 3.2e-4 / 3.7e-5 (RBC-642 / PLT-162)
        assert rel_l2(xs[t] - x0, xr - x0) <= (TOL_FP64 if precision == "fp64" else 1.5e-4)
        assert rel_l2(vs[t], vr) <= (TOL_FP64 if precision == "fp64" else 6.5e-4)
        assert np.linalg.norm(vs[t], axis=-1).max() <= v_max * (1 + 1e-6)


@pytest.mark.parametrize("precision,where", [("fp64", "device"), ("fp32", "host")])
def test_collision_term_matches_oracle(precision, where):
    """PIK collision energy 1/2 k |x - p|^2 on flagged vertices in the
    gradient and in the objective, mixed cell types, a subset of the cells in contact."""
    import torch
    from oracle import npfem_oracle as orc
    from paper_1911_03062_b200 import Solver, binding
    pop = make_config(3, n_cells=23)
    rng = np.random.default_rng(31)
    n_steps, n_its = 2, 6
    targets, stiff = [], []
    for t, ct in enumerate(pop.types):
        k = np.where(rng.random(pop.positions[t].shape[:2]) < 0.15, rng.uniform(20, 300, pop.positions[t].shape[:2]), 0.0)
        k[::2] = 0.0                                              # every other cell is not in contact at all
        targets.append(pop.positions[t] + 0.02 * rng.standard_normal(pop.positions[t].shape))
        stiff.append(k)
    np_io = np.float64 if precision == "fp64" else np.float32
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision=precision)
    solver.set_option(binding.OPT_DIAGNOSTICS, 1)
    solver.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
    tg, kk = pop.packed(targets), pop.packed([k[..., None].repeat(3, -1) for k in stiff])[::3].copy()
    if where == "device":
        solver.set_collisions(torch.from_numpy(tg).cuda(), torch.from_numpy(kk).cuda())
    else:
        solver.set_collisions(tg.astype(np.float64), kk.astype(np.float64))
    for s in range(n_steps):
        solver.set_forces(torch.from_numpy(pop.packed(pop.forces(s), dtype=np_io)).cuda())
        solver.step(n_its)
    x, v = solver.get_state()
    hist, mono = solver.get_objective()
    xs = pop.unpack(x.cpu().numpy())
    for t, ct in enumerate(pop.types):
        td = orc.make_type(ct, pop.dt)
        col = (targets[t], stiff[t])
        xr, vr = orc.run(pop.positions[t], pop.velocities[t], lambda s, t=t: pop.forces(s)[t], td, n_steps, n_its, collisions=col)
        x_plain, _ = orc.run(pop.positions[t], pop.velocities[t], lambda s, t=t: pop.forces(s)[t], td, n_steps, n_its)
        x0 = pop.positions[t]
        assert rel_l2(xr - x0, x_plain - x0) > 0.05               # the contacts matter
        print(precision, ct.name, rel_l2(xs[t], xr), rel_l2(xs[t] - x0, xr - x0))
        assert rel_l2(xs[t], xr) <= TOL_POS[precision]
        assert rel_l2(xs[t] - x0, xr - x0) <= (TOL_FP64 if precision == "fp64" else 2.8e-4)   # fp32 measured 1.4e-4 / 6.6e-5
    # objective of the last step (diagnostics) includes the collision energy
    t = 0
    td = orc.make_type(pop.types[t], pop.dt)
    xr1, vr1 = orc.run(pop.positions[t], pop.velocities[t], lambda s: pop.forces(s)[t], td, 1, n_its, collisions=(targets[t], stiff[t]))
    _, _, rec = orc.step(xr1, vr1, pop.forces(1)[t], td, n_its, record=True, collisions=(targets[t], stiff[t]))
    ref = np.array(rec["objective"])
    ids = np.nonzero(pop.type_of_cell == t)[0]
    scale = np.abs(ref).max()
    assert np.abs(hist[:, ids] - ref).max() < (1e-8 if precision == "fp64" else 5e-3) * scale
    # clearing restores the plain step
    solver.clear_collisions()
    solver.close()


@pytest.mark.parametrize("config,cells,fused", [(6, None, 2), (6, None, 0), (6, 700, 2)])
def test_whole_step_fused_kernel(config, cells, fused):
    """the small-batch path, one kernel per time step and one CTA per cell (prologue, K
    iterations with the per-cell FP32 product by H~^-1, epilogue), against the oracle: the paper's own
    load (config 6: forced and auto-selected; 700 cells: several cells per CTA), forces redrawn every step.
    (Types above 256 threads per cell, e.g. RBC-642, always take the batched kernels.)"""
    pop = make_config(config, n_cells=cells)
    gpu, solver = run_gpu(pop, "fp32", n_steps=4, n_iterations=5, fused_step=fused)
    times = solver.get_kernel_times(reset=False)
    solver.close()
    ref = run_oracle(pop, 4, 5)
    for r in compare(pop, gpu, ref):
        print(config, fused, r)
        # measured RBC-258 1.7e-4, 3.1e-4, 9.8e-4, 4.0e-4; PLT-66 4.5e-5, 4.0e-4, 8.1e-4, 1.2e-4 (round 1: 1.0e-3 / 2.0e-3,
        # the floor of a one-float state: DESIGN.md section 5)
        assert_row(r, "fp32", (3.4e-4, 8e-4, 2e-3, 8e-4))


def test_whole_step_fused_kernel_is_the_one_that_ran():
    """The fused path really replaces the batched launches: 1 launch per type and step."""
    import torch
    from paper_1911_03062_b200 import Solver, binding
    pop = make_config(6)
    for fused, per_step in ((2, 2), (1, 2 * (2 + 2 * 5))):
        solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision="fp32")
        solver.set_option(binding.OPT_FUSED_STEP, fused)
        solver.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
        solver.set_forces(torch.from_numpy(pop.packed(pop.forces(0))).cuda())
        before = solver.launch_count
        solver.step(5)
        assert solver.launch_count - before == per_step
        solver.close()


@pytest.mark.parametrize("precision", ["fp32", "fp64"])
def test_paper_resolution_meshes_config6(precision):
    """the paper's own resolutions (octahedral RBC-258 / PLT-66), its
    per-GPU load of 114 cells and h = 0.25 us; valence-4 vertices, 2 overflow vertices on a 256-thread CTA."""
    pop = make_config(6)
    assert [ct.n_vertices for ct in pop.types] == [258, 66] and pop.n_cells == 114 and pop.dt == 0.25
    # batched kernels (114 cells: auto would take the whole-step kernel; run_gpu forces the batched path)
    # measured RBC-258 2.0e-4, 3.5e-4, 1.1e-3, 4.2e-4; PLT-66 1.5e-4, 9.5e-4, 1.7e-3, 2.0e-4
    _check(pop, precision, fp32=(4e-4, 1.9e-3, 3.5e-3, 8.4e-4), n_steps=4, n_iterations=5)


def _sampled_full_size(config, precision, n_steps, n_iterations, samples_per_type=6):
    """BASELINE.json full size in the launch configuration bench.py times; the oracle recomputes a seeded
    sample of cells one by one (cells are independent: PAPER.md:61, :63), first and last slot included."""
    import torch
    from oracle import npfem_oracle as orc
    from paper_1911_03062_b200 import Solver
    pop = make_config(config)
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision=precision)
    solver.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
    np_io = np.float32 if precision == "fp32" else np.float64
    for s in range(n_steps):
        solver.set_forces(torch.from_numpy(pop.packed(pop.forces(s), dtype=np_io)).cuda())
        solver.step(n_iterations)
    rng = np.random.default_rng(100 + config)
    rows = []
    for t, ct in enumerate(pop.types):
        ids = pop.cells_of_type(t)
        if ids.size == 0:
            continue
        slots = np.unique(np.concatenate(([0, ids.size - 1], rng.integers(0, ids.size, samples_per_type))))
        x, v = solver.get_state(cell_ids=ids[slots])
        xg = x.cpu().numpy().reshape(slots.size, ct.n_vertices, 3)
        vg = v.cpu().numpy().reshape(slots.size, ct.n_vertices, 3)
        td = orc.make_type(ct, pop.dt)
        x0 = pop.positions[t][slots]
        xr, vr = orc.run(x0, pop.velocities[t][slots], lambda s, t=t: pop.forces(s)[t][slots], td, n_steps, n_iterations)
        rows.append((ct.name, rel_l2(xg, xr), rel_l2(xg - x0, xr - x0), rel_l2(vg, vr)))
    solver.close()
    return rows


def test_full_size_config4_100k_cells_sampled():
    """BASELINE configs[3] at its full 100,000 cells, fp32, default kernels (what bench.py times); the oracle
    recomputes a seeded sample of ~1,000 cells per type, about a minute of host time."""
    for name, pos, disp, vel in _sampled_full_size(4, "fp32", n_steps=2, n_iterations=10, samples_per_type=1000):
        print(name, pos, disp, vel)
        assert pos <= TOL_POS["fp32"] and disp <= 1.2e-4 and vel <= 1.4e-4      # measured 5.6e-5 / 2.5e-5 and 7.0e-5 / 2.7e-5


@pytest.mark.parametrize("precision", ["fp32", "fp64"])
def test_full_size_config5_10k_level4_cells_sampled(precision):
    """BASELINE configs[4] at its full 10,000 RBC-2562 cells (generic local step, 11-pass GEMM)."""
    for name, pos, disp, vel in _sampled_full_size(5, precision, n_steps=1, n_iterations=5, samples_per_type=3):
        print(name, pos, disp, vel)
        bound = TOL_FP64 if precision == "fp64" else 5.6e-4                       # fp32 measured 2.8e-4 (disp = vel: one step)
        assert pos <= TOL_POS[precision] and disp <= bound and vel <= bound


@pytest.mark.parametrize("kappa", [0.7, 0.8, 0.9])
def test_kappa_damping_sweep_config6(kappa):
    """the paper's parameter sweep kappa_damping in {0.5, 0.7, 0.8, 0.9} on its
    own meshes; 0.5 is the default of every other test.  Batched kernels in fp64, whole-step kernel in fp32."""
    import dataclasses
    pop = make_config(6, n_cells=36)
    pop.types = [dataclasses.replace(ct, material=dataclasses.replace(ct.material, kappa_damping=kappa))
                 for ct in pop.types]
    _check(pop, "fp64", n_steps=5, n_iterations=5)
    # measured (all three kappa): RBC-258 1.3e-4, 3.0e-4, 1.1e-3, 3.7e-4; PLT-66 3.5e-5, 7.5e-5, 2.1e-4, 1.3e-4
    _check(pop, "fp32", fp32=(2.6e-4, 6.1e-4, 2.2e-3, 7.5e-4), n_steps=5, n_iterations=5, fused_step=2)


@pytest.mark.parametrize("precision", ["fp32", "fp64"])
def test_static_partition_shards_match_the_unsharded_solver(precision):
    """cells are independent within a step, so the shards of a
    static partition, each stepped by its own solver (here one after the other on the one GPU there is),
    reproduce the unsharded run bit for bit, whatever the batch a cell finds itself in."""
    import torch
    from paper_1911_03062_b200 import Solver, binding
    from paper_1911_03062_b200.partition import ShardedSolver
    pop = make_config(3, n_cells=45)
    x0 = pop.packed(pop.positions)
    forces = [pop.packed(pop.forces(s)) for s in range(3)]

    def factory(types, toc, dt):
        s = Solver(types, toc, dt, precision=precision)
        s.set_option(binding.OPT_FUSED_STEP, 1)
        return s

    whole = ShardedSolver(pop.types, pop.type_of_cell, pop.dt, 0, 1, solver_factory=factory)
    shards = [ShardedSolver(pop.types, pop.type_of_cell, pop.dt, r, 3, solver_factory=factory) for r in range(3)]
    assert sorted(int(c) for s in shards for c in s.cell_ids) == list(range(pop.n_cells))
    for s in [whole] + shards:
        s.set_state(x0)
        for f in forces:
            s.set_forces(f)
            s.step(5)
    torch.cuda.synchronize()
    xw, vw = whole.gather_state()
    part = shards[0].partition
    xs = part.assemble([s.local_state()[0] for s in shards])
    vs = part.assemble([s.local_state()[1] for s in shards])
    assert np.array_equal(xs, xw) and np.array_equal(vs, vw)
    assert np.linalg.norm(xw - x0) > 0
    for s in [whole] + shards:
        s.solver.close()


@pytest.mark.parametrize("precision,n_chunks", [("fp32", 7), ("fp32", 0), ("fp64", 4), ("fp32", 64)])
def test_step_host_pipelined_equals_the_three_calls(precision, n_chunks):
    """npfem_step_host (include/npfem.h): forces in, step, state out over chunks of cell ids on copy streams.
    Chunks are contiguous slabs of every bucket, cells are independent: bit-identical to
    set_forces + step + get_state, with ragged chunk sizes, interleaved types and more chunks than PLT cells."""
    import torch
    from paper_1911_03062_b200 import Solver, binding
    pop = make_config(3, n_cells=45)
    np_io = np.float32 if precision == "fp32" else np.float64
    x0 = pop.packed(pop.positions, dtype=np_io)
    out = []
    for pipelined in (False, True):
        s = Solver(pop.types, pop.type_of_cell, pop.dt, precision=precision)
        s.set_option(binding.OPT_FUSED_STEP, 1)
        s.set_state(x0)
        x = torch.empty(x0.size, dtype=torch.from_numpy(x0[:1]).dtype).pin_memory()
        v = torch.empty_like(x).pin_memory()
        for k in range(3):
            f = torch.from_numpy(pop.packed(pop.forces(k), dtype=np_io)).pin_memory()
            if pipelined:
                s.step_host(f, 5, x, v, n_chunks=n_chunks)
            else:
                s.set_forces(f)
                s.step(5)
                s.get_state(positions=x, velocities=v)
        out.append((x.numpy().copy(), v.numpy().copy()))
        s.close()
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    assert np.linalg.norm(out[0][0] - x0) > 0 and np.all(np.isfinite(out[0][1]))


def test_step_host_with_line_search_takes_the_unchunked_sequence():
    import torch
    from paper_1911_03062_b200 import Solver
    pop = make_config(2, n_cells=6)
    x0 = pop.packed(pop.positions)
    f = torch.from_numpy(pop.packed(pop.forces(0))).pin_memory()
    res = []
    for pipelined in (False, True):
        s = Solver(pop.types, pop.type_of_cell, pop.dt, precision="fp64")
        s.set_line_search(3)
        s.set_state(x0)
        x = torch.empty(x0.size, dtype=torch.float64).pin_memory()
        v = torch.empty_like(x).pin_memory()
        if pipelined:
            s.step_host(f, 4, x, v, n_chunks=3)
        else:
            s.set_forces(f); s.step(4); s.get_state(positions=x, velocities=v)
        res.append(x.numpy().copy())
        s.close()
    assert np.array_equal(res[0], res[1])


def test_full_size_config4_momentum_balance_every_cell():
    """Pin P4 as a property that holds at any size, over ALL 100,000 cells of BASELINE
    configs[3] in the launch configuration bench.py times: 1^T L = 0, so with v_0 = 0 and a constant force
    the mass centre of every cell after N steps sits at h^2 (sum F / sum m) N (N + 1) / 2, whatever the
    stiffness, damping (kappa, beta) or iteration count.  fp32 state + TF32 operator: the balance holds
    to the rounding of the increment, measured against the cell's own displacement scale."""
    import torch
    from oracle import npfem_oracle as orc
    from paper_1911_03062_b200 import Solver
    pop = make_config(4)
    n_steps, n_iterations = 4, 10
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision="fp32")
    solver.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
    solver.set_forces(torch.from_numpy(pop.packed(pop.forces(0), dtype=np.float32)).cuda())
    for _ in range(n_steps):
        solver.step(n_iterations)
    x, v = solver.get_state()
    xs = pop.unpack(x.cpu().numpy())
    vs = pop.unpack(v.cpu().numpy())
    solver.close()
    forces = pop.forces(0)
    for t, ct in enumerate(pop.types):
        m = orc.make_type(ct, pop.dt).mass                               # [n] lumped masses, fg
        acc = forces[t].sum(axis=1) / m.sum()                            # [cells, 3] um / us^2
        expect = pop.dt ** 2 * acc * n_steps * (n_steps + 1) / 2
        got = np.einsum("i,cik->ck", m, xs[t] - pop.positions[t]) / m.sum()
        vexp = pop.dt * acc * n_steps                                    # and the momentum itself
        vgot = np.einsum("i,cik->ck", m, vs[t]) / m.sum()
        scale = np.linalg.norm(expect, axis=1).max()
        err = np.linalg.norm(got - expect, axis=1).max() / scale
        verr = np.linalg.norm(vgot - vexp, axis=1).max() / np.linalg.norm(vexp, axis=1).max()
        print(ct.name, "cells", xs[t].shape[0], "centre err", err, "momentum err", verr, "scale um", scale)
        assert err <= 5e-5 and verr <= 5e-5      # measured 9e-6 (1.3e-4 before both GEMM operands were rounded to TF32 to nearest)


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_level5_mesh_10242_vertices_runs_from_global_scratch(precision):
    """Maximum size: a level-5 icosphere cell (10,242 vertices, 20,480 triangles, H~^-1 of 10,256^2).  None of
    the shared-memory local-step kernels can hold it; the generic kernel keeps the cell in a per-CTA slab of
    global scratch.  One cell, 1 step x 3 iterations against the oracle."""
    pop = make_config(1, level=5)
    assert pop.types[0].n_vertices == 10242
    _check(pop, precision, fp32=(5.1e-4, 5.1e-4, 1.7e-3, 5.1e-4), n_steps=1, n_iterations=3)   # measured 2.5e-4, 2.5e-4, 8.4e-4, 2.5e-4


@pytest.mark.parametrize("precision", ["fp32", "fp64"])
def test_drifting_cells_recentre_their_local_frame(precision):
    """state lives in cell-local coordinates and the prologue shifts a cell's frame by an exact
    binary amount once its mass centre has drifted by more than 0.5 um.  A steady 20 pN push per vertex moves
    every cell by ~2.4 um in 60 steps (several shifts); the run must still match the oracle and the closed-form
    mass-centre trajectory of pin P4."""
    import torch
    from oracle import npfem_oracle as orc
    from paper_1911_03062_b200 import Solver, binding
    pop = make_config(3, n_cells=12)
    n_steps, n_iterations = 60, 3
    forces = [f.copy() for f in pop.forces(0)]
    for f in forces:
        f[..., 0] += 20.0
    np_io = np.float32 if precision == "fp32" else np.float64
    solver = Solver(pop.types, pop.type_of_cell, pop.dt, precision=precision)
    solver.set_option(binding.OPT_FUSED_STEP, 1)
    solver.set_state(torch.from_numpy(pop.packed(pop.positions)).cuda())
    solver.set_forces(torch.from_numpy(pop.packed(forces, dtype=np_io)).cuda())
    for _ in range(n_steps):
        solver.step(n_iterations)
    x, v = solver.get_state()
    xs, vs = pop.unpack(x.cpu().numpy()), pop.unpack(v.cpu().numpy())
    solver.close()
    for t, ct in enumerate(pop.types):
        td = orc.make_type(ct, pop.dt)
        xr, vr = orc.run(pop.positions[t], pop.velocities[t], lambda s, t=t: forces[t], td, n_steps, n_iterations)
        disp, vel = rel_l2(xs[t] - pop.positions[t], xr - pop.positions[t]), rel_l2(vs[t], vr)
        centre = np.einsum("i,cik->ck", td.mass, xs[t] - pop.positions[t]) / td.mass.sum()
        expect = pop.dt ** 2 * forces[t].sum(axis=1) / td.mass.sum() * n_steps * (n_steps + 1) / 2
        cerr = np.linalg.norm(centre - expect, axis=1).max() / np.linalg.norm(expect, axis=1).max()
        print(precision, ct.name, "disp", disp, "vel", vel, "centre", cerr, "moved um", np.linalg.norm(expect, axis=1).min())
        assert np.linalg.norm(expect, axis=1).min() > 2.0               # far beyond the 0.5 um threshold
        assert disp <= (3.3e-5 if precision == "fp32" else TOL_FP64) and vel <= (3.6e-5 if precision == "fp32" else TOL_FP64)   # fp32 measured 1.6e-5 / 1.8e-5
        assert cerr <= (2.3e-5 if precision == "fp32" else 1e-9)     # fp32: measured 1.1e-5 (1.3e-3 with truncated TF32 operands)


@pytest.mark.parametrize("cells", [600, 1800])
def test_step_host_chunks_take_the_kernels_of_the_whole_bucket(cells):
    """The whole-step kernel is chosen by bucket size (<= 1.5 cells per SM).  600 cells of config 6: the PLT-66 bucket
    (100 cells) takes it, so npfem_step_host does not chunk; 1,800 cells: no bucket takes it, and no CHUNK (75 PLT
    cells) may either - both ways the result is bit-identical to the three calls."""
    import torch
    from paper_1911_03062_b200 import Solver
    pop = make_config(6, n_cells=cells)
    x0 = pop.packed(pop.positions, dtype=np.float32)
    f = torch.from_numpy(pop.packed(pop.forces(0), dtype=np.float32)).pin_memory()
    out = []
    for pipelined in (False, True):
        s = Solver(pop.types, pop.type_of_cell, pop.dt, precision="fp32")
        s.set_state(x0)
        x = torch.empty(x0.size, dtype=torch.float32).pin_memory()
        v = torch.empty_like(x).pin_memory()
        for _ in range(2):
            if pipelined:
                s.step_host(f, 5, x, v, n_chunks=4)
            else:
                s.set_forces(f); s.step(5); s.get_state(positions=x, velocities=v)
        out.append((x.numpy().copy(), v.numpy().copy()))
        s.close()
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
