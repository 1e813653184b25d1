"""Host logic of the scheduled local step (no GPU): the create-time shared-memory schedule
(paper_1911_03062_b200/csrc/local_schedule.hpp) through the C-ABI diagnostic
npfem_local_schedule_stats.  The library decodes its own tables and checks them against the mesh;
these tests pin the properties the kernel relies on."""
import dataclasses

import numpy as np
import pytest

from paper_1911_03062_b200.binding import local_schedule_stats, NpfemError
from workloads import icosahedron_cell_type
from workloads.meshes import irregular_cell_type, platelet_cell_type, rbc_cell_type


@pytest.mark.parametrize("make,threads,tpt", [(lambda: rbc_cell_type(3), 640, 2), (lambda: platelet_cell_type(2), 320, 1),
                                              (lambda: icosahedron_cell_type(3.0), 32, 1)])
def test_schedule_of_the_baseline_cell_types(make, threads, tpt):
    st = local_schedule_stats(make(), 0.1)
    assert st["valid"] == 1 and st["threads"] == threads and st["triangles_per_thread"] == tpt
    assert st["tables_consistent"] == 1
    # corner forces: exact bipartite edge colouring -> stores and gathers are conflict-free
    assert st["worst_corner_store"] == 1 and st["worst_corner_gather"] == 1
    # vertex / normal gathers: min-conflicts colouring, ideal is 4 wavefronts per LDS.128
    assert 4.0 <= st["wavefronts_vertex_gather"] <= 4.6
    assert 4.0 <= st["wavefronts_normal_gather"] <= 5.2
    assert st["smem_bytes"] < 100 * 1024


def test_schedule_of_an_irregular_mesh():
    ct = irregular_cell_type(2, 40, seed=3)
    val = np.bincount(ct.triangles.ravel())
    assert val.min() >= 4 and val.max() in (7, 8)            # needs the 8-read variant of the kernel
    st = local_schedule_stats(ct, 0.1)
    assert st["valid"] == 1 and st["tables_consistent"] == 1
    assert st["worst_corner_store"] == 1 and st["worst_corner_gather"] == 1


def test_schedule_rejects_what_the_kernel_cannot_hold():
    st = local_schedule_stats(rbc_cell_type(4), 0.1)          # 5120 triangles: generic kernel instead
    assert st["valid"] == 0
    bad = rbc_cell_type(2)
    bad = dataclasses.replace(bad, triangles=bad.triangles[:-1])      # open surface
    with pytest.raises(NpfemError) as e:
        local_schedule_stats(bad, 0.1)
    assert e.value.code == -2


def test_schedule_is_deterministic():
    a, b = local_schedule_stats(rbc_cell_type(2), 0.1), local_schedule_stats(rbc_cell_type(2), 0.1)
    a.pop("build_ms"), b.pop("build_ms")
    assert a == b


# ---- quad local step (one thread per pair of adjacent triangles; csrc/quad_schedule.hpp) --------------------------
from paper_1911_03062_b200.binding import quad_schedule_stats  # noqa: E402


@pytest.mark.parametrize("make,threads", [(lambda: rbc_cell_type(3), 640), (lambda: platelet_cell_type(2), 160),
                                          (lambda: rbc_cell_type(3, base="octa"), 256),
                                          (lambda: platelet_cell_type(2, base="octa"), 64)])
def test_quad_schedule_of_the_baseline_and_paper_cell_types(make, threads):
    """A perfect matching of the dual graph exists for these meshes (T even, bridgeless cubic graph: Petersen), the
    tables decode to the mesh's connectivity, and the corner-force traffic is conflict-free."""
    st = quad_schedule_stats(make(), 0.1)
    assert st["valid"] == 1 and st["threads"] == threads and st["consistent"] == 1
    assert st["reads_per_vertex"] == 6                      # every vertex lies in at most 6 quads (of its <= 6 triangles)
    assert st["worst_store_quarter"] == 1 and st["worst_gather_quarter"] == 1
    assert 4.0 <= st["wf_vertex_gather"] <= 6.0 and 4.0 <= st["wf_normal_gather"] <= 6.0
    assert st["smem_bytes"] < 100 * 1024


def test_quad_schedule_irregular_mesh_and_rejections():
    st = quad_schedule_stats(irregular_cell_type(2, 40, seed=3), 0.1)       # valence up to 8
    assert st["valid"] == 1 and st["consistent"] == 1
    assert st["worst_store_quarter"] == 1 and st["worst_gather_quarter"] == 1
    assert quad_schedule_stats(rbc_cell_type(4), 0.1)["valid"] == 0          # 5,120 triangles: other kernels
    a, b = quad_schedule_stats(rbc_cell_type(2), 0.1), quad_schedule_stats(rbc_cell_type(2), 0.1)
    a.pop("build_ms"), b.pop("build_ms")
    assert a == b                                                            # deterministic


def test_multipass_quad_schedule_of_the_level4_mesh():
    """RBC-2562 (BASELINE configs[4]): 2,560 quads in 4 passes of 640; global vertex / normal slots, per-pass corner
    slots and per-pass vertex lists, all decoded and checked against the mesh by the library."""
    st = quad_schedule_stats(rbc_cell_type(4), 0.1, multipass=True)
    assert st["valid"] == 1 and st["threads"] == 4 and st["consistent"] == 1      # "threads" = passes here
    assert st["reads_per_vertex"] == 6
    assert st["worst_store_quarter"] == 1 and st["worst_gather_quarter"] == 1
    assert 4.0 <= st["wf_vertex_gather"] <= 6.0 and 4.0 <= st["wf_normal_gather"] <= 6.0
    assert st["smem_bytes"] <= 227 * 1024
    # 1,024 quads: one full pass and one of 384 (threads without a quad in the last pass)
    st2 = quad_schedule_stats(rbc_cell_type(4, base="octa"), 0.1, multipass=True)
    assert st2["valid"] == 1 and st2["threads"] == 2 and st2["consistent"] == 1
    assert st2["worst_store_quarter"] == 1 and st2["worst_gather_quarter"] == 1
    # one pass suffices for the smaller meshes (the one-pass kernel takes them); too many passes are refused
    assert quad_schedule_stats(rbc_cell_type(3), 0.1, multipass=True)["threads"] == 1
    assert quad_schedule_stats(rbc_cell_type(5), 0.1, multipass=True)["valid"] == 0
