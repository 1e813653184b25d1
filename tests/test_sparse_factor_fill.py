"""Pins the numbers behind a design decision (SURVEY.md section 7 "compare against a sparse-factor
solve before committing"): the fill of a sparse Cholesky-type factor of the constant H~ of Eq. (4)
and therefore the flops of a sparse triangular solve per cell and iteration, against the 6 n^2 of the dense apply
the CUDA path uses.  CPU only (scipy SuperLU, minimum-degree ordering on A^T + A, no pivoting: H~ is SPD)."""
import numpy as np
import pytest
import scipy.sparse as sp
import scipy.sparse.linalg as spla

from oracle import npfem_oracle as orc
from workloads.meshes import rbc_cell_type


@pytest.mark.parametrize("level,n,ratio_lo,ratio_hi", [(3, 642, 4.5, 5.7), (4, 2562, 11.5, 14.0)])
def test_sparse_factor_fill_vs_dense_apply(level, n, ratio_lo, ratio_hi):
    td = orc.make_type(rbc_cell_type(level), 0.1)
    H = td.H_tilde
    assert H.shape == (n, n)
    Hs = sp.csc_matrix(np.where(np.abs(H) > 1e-14 * np.abs(H).max(), H, 0.0))
    assert 18.0 < Hs.nnz / n < 20.0                        # two-ring stencil of the bi-Laplacian: ~19 entries per row
    lu = spla.splu(Hs, permc_spec="MMD_AT_PLUS_A", diag_pivot_thresh=0.0, options=dict(SymmetricMode=True))
    solve_flops = 2 * 2 * lu.L.nnz * 3                      # forward + backward substitution, 3 coordinate columns
    dense_flops = 6 * n * n
    ratio = dense_flops / solve_flops
    print(f"n = {n}: nnz(L) = {lu.L.nnz}, sparse solve {solve_flops / 1e6:.2f} MFLOP, dense apply {dense_flops / 1e6:.2f} MFLOP, "
          f"ratio {ratio:.1f}")
    assert ratio_lo < ratio < ratio_hi
    # the factor really solves the system (the permutations are the factor's own)
    rhs = np.random.default_rng(0).standard_normal((n, 3))
    assert np.allclose(H @ lu.solve(rhs), rhs, rtol=1e-9, atol=1e-9 * np.abs(rhs).max())
