"""npfem_invert_spd_static (include/npfem.h): the entry point that allocates nothing - its scratch is a file-scope
`static __device__` array inside the library (paper_1911_03062_b200/csrc/inverse_static.cu).

Collected LAST on purpose (file name): the suite runs with `pytest -x`, a failure here must not hide other tests.
The matrices are H~ = M~/h^2 + L of the paper's own resolutions (RBC 258 / platelet 66 vertices),
built by the oracle: 258 is exactly NPFEM_INVERT_STATIC_MAX_N.  The existing path is npfem_invert_spd, the same
Newton-Schulz chain npfem_create runs, with caller-owned scratch."""
import numpy as np
import pytest

from workloads import make_config

pytestmark = pytest.mark.gpu

TOL_FP64 = 1e-8          # the fp64 tolerance of tests/test_parity_gpu.py


def _h_tilde(pop):
    from oracle import npfem_oracle as orc
    return [np.ascontiguousarray(orc.make_type(ct, pop.dt).H_tilde, dtype=np.float64) for ct in pop.types]


def _rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def test_static_scratch_inverse_matches_the_existing_path_twice_in_a_row_without_allocating():
    import torch
    from paper_1911_03062_b200 import binding
    assert binding.INVERT_STATIC_MAX_N == 258
    h_rbc, h_plt = _h_tilde(make_config(6, n_cells=6))
    assert h_rbc.shape == (258, 258) and h_plt.shape == (66, 66)
    mats = [torch.from_numpy(h).cuda() for h in (h_rbc, h_plt)]
    # existing path: caller-owned scratch (torch's memory), the chain npfem_create runs
    ref = []
    for H in mats:
        inv, res = binding.invert_spd(H)
        assert res <= 1e-13 * np.sqrt(H.shape[0]) or res < 1e-9
        ref.append(inv.cpu().numpy())
    # and that path is an inverse at all (plain definition, LAPACK on the host)
    for h, r in zip((h_rbc, h_plt), ref):
        assert _rel(r, np.linalg.inv(h)) <= TOL_FP64
        assert np.abs(r @ h - np.eye(h.shape[0])).max() <= 1e-10
    # two calls in a row on the shared array: the large matrix first, so that the second call (n = 66) starts on a
    # scratch full of the first one's iterates; then the large one again on what the small one left behind
    order = (0, 1, 0)
    outs = [torch.full_like(mats[i], float("nan")) for i in order]
    binding.invert_spd_static(mats[1], torch.empty_like(mats[1]))   # loads the module / asks the symbol address once
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info(0)
    residuals = [binding.invert_spd_static(mats[i], out) for i, out in zip(order, outs)]   # library calls only
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info(0)
    assert free_after == free_before, (free_before, free_after)
    for i, out, res in zip(order, outs, residuals):
        assert res < 1e-9
        got = out.cpu().numpy()
        assert np.isfinite(got).all()
        assert _rel(got, ref[i]) <= TOL_FP64, _rel(got, ref[i])
        assert np.array_equal(got, got.T)                      # symmetrised like the existing path


def test_static_scratch_inverse_refuses_sizes_beyond_its_maximum_and_bad_arguments():
    import torch
    from paper_1911_03062_b200 import binding
    n = binding.INVERT_STATIC_MAX_N + 1
    H = torch.eye(n, dtype=torch.float64, device="cuda:0") * 3.0
    out = torch.zeros_like(H)
    with pytest.raises(binding.NpfemError) as e:
        binding.invert_spd_static(H, out)
    assert e.value.code == -1 and "NPFEM_INVERT_STATIC_MAX_N = 258" in str(e.value)
    assert float(out.abs().max()) == 0.0                       # nothing was launched
    # the caller-owned variant takes the same size
    inv, _ = binding.invert_spd(H)
    assert torch.allclose(inv, torch.eye(n, dtype=torch.float64, device="cuda:0") / 3.0, rtol=0, atol=1e-15)
    # not SPD: refused with a message, not a wrong answer
    bad = torch.eye(8, dtype=torch.float64, device="cuda:0")
    bad[3, 3] = -1.0
    with pytest.raises(binding.NpfemError) as e:
        binding.invert_spd_static(bad, torch.empty_like(bad))
    assert e.value.code == -1 and "SPD" in str(e.value)
    lib = binding.load_library()
    assert lib.npfem_invert_spd_static(None, None, 4, None, None) == -1
    assert lib.npfem_invert_spd_tmp_bytes(258) == (3 * 258 * 258 + 32) * 8
