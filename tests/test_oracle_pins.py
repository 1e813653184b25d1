"""Pins of the fp64 oracle against what the paper and the mathematics fix.

P1..P13 are the pins of SURVEY.md section 8(c); each is chosen so that a plausible
mistake in oracle/npfem_oracle.py (dropped term, wrong sign/index, transposed
operand) fails at least one.  CPU only.
"""
import copy
import math
import os

import numpy as np
import pytest
import scipy.integrate
import scipy.optimize

from oracle import npfem_oracle as orc
from workloads import (icosahedron_cell_type, icosphere, platelet_cell_type, rbc_cell_type)
from workloads.meshes import Material

H = 0.1  # us (BASELINE.json dt = 1e-7 s)
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rotation(rng):
    q = rng.standard_normal(4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


@pytest.fixture(scope="module")
def ico():
    ct = icosahedron_cell_type(3.0)
    return ct, orc.make_type(ct, H)


@pytest.fixture(scope="module")
def rbc162():
    ct = rbc_cell_type(2)
    return ct, orc.make_type(ct, H)


@pytest.fixture(scope="module")
def rbc642():
    ct = rbc_cell_type(3)
    return ct, orc.make_type(ct, H)


# ---- P1 ------------------------------------------------------------------------------
def test_p1_rest_state_no_force_no_motion(rbc642):
    ct, td = rbc642
    rng = np.random.default_rng(11)
    x = ct.rest_positions @ _rotation(rng).T + rng.uniform(0, 100, 3)
    # round-off only: k_mem ~ 1e4 pN/um times ulp(100 um) ~ 1.4e-14 um per edge of 0.5 um
    assert np.abs(orc.grad_energy(x, td)).max() < 2e-9
    assert np.abs(orc.grad_energy(ct.rest_positions, td)).max() < 1e-11
    x1, v1 = orc.step(x, np.zeros_like(x), np.zeros_like(x), td, 5)
    assert np.abs(x1 - x).max() < 1e-12
    assert np.abs(v1).max() < 1e-11


# ---- P2 ------------------------------------------------------------------------------
@pytest.mark.parametrize("fixture", ["ico", "rbc162"])
def test_p2_rigid_motion_invariance_and_momenta(fixture, request):
    ct, td = request.getfixturevalue(fixture)
    rng = np.random.default_rng(5)
    x = ct.rest_positions + 0.05 * rng.standard_normal(ct.rest_positions.shape)
    Q, t = _rotation(rng), rng.uniform(-20, 20, 3)
    xq = x @ Q.T + t
    e0 = orc.energies(x, td)
    e1 = orc.energies(xq, td)
    for k in e0:
        assert e1[k] == pytest.approx(e0[k], rel=1e-9, abs=1e-12), k
    g = orc.grad_energy(x, td)
    gq = orc.grad_energy(xq, td)
    scale = np.abs(g).max()
    assert scale > 1e-3                                   # the state is genuinely deformed
    assert np.abs(gq - g @ Q.T).max() < 1e-8 * scale
    assert np.abs(g.sum(axis=0)).max() < 1e-9 * scale           # sum F_int = 0
    assert np.abs(np.cross(x, g).sum(axis=0)).max() < 1e-8 * scale   # sum x x F_int = 0
    for grad in (orc.grad_membrane, orc.grad_bending, orc.grad_volume):
        gi = grad(x, td)
        assert np.abs(gi.sum(axis=0)).max() < 1e-9 * max(np.abs(gi).max(), 1e-30)


# ---- P3 ------------------------------------------------------------------------------
@pytest.mark.parametrize("fixture", ["ico", "rbc162"])
@pytest.mark.parametrize("family", ["strain", "area", "bend", "volume"])
def test_p3_finite_difference_gradients(fixture, family, request):
    ct, td = request.getfixturevalue(fixture)
    rng = np.random.default_rng(7)
    x = ct.rest_positions + 0.03 * rng.standard_normal(ct.rest_positions.shape)
    td1 = copy.copy(td)
    # isolate one family by zeroing the constants of the others
    if family == "strain":
        td1.C, td1.k_b, td1.k_v = 0.0, 0.0, 0.0
    elif family == "area":
        td1.B, td1.k_b, td1.k_v = 0.0, 0.0, 0.0
    elif family == "bend":
        td1.B, td1.C, td1.k_v = 0.0, 0.0, 0.0
    else:
        td1.B, td1.C, td1.k_b = 0.0, 0.0, 0.0
    analytic = orc.grad_energy(x, td1)
    assert np.abs(analytic).max() > 0
    eps = 1e-6
    idx = rng.choice(x.shape[0], size=min(12, x.shape[0]), replace=False)
    for v in idx:
        for c in range(3):
            xp, xm = x.copy(), x.copy()
            xp[v, c] += eps
            xm[v, c] -= eps
            fd = (orc.energies(xp, td1)[family] - orc.energies(xm, td1)[family]) / (2 * eps)
            assert fd == pytest.approx(analytic[v, c], rel=2e-6, abs=1e-7 * np.abs(analytic).max())


# ---- P4 ------------------------------------------------------------------------------
@pytest.mark.parametrize("kappa", [0.0, 0.5])
def test_p4_momentum_balance_closed_form(rbc162, kappa):
    ct, td0 = rbc162
    td = copy.copy(td0)
    td.kappa = kappa
    rng = np.random.default_rng(3)
    x = ct.rest_positions.copy()
    v = np.zeros_like(x)
    F = rng.standard_normal(x.shape) + np.array([0.3, -0.2, 0.1])
    m = td.mass
    cm0 = (m[:, None] * x).sum(0) / m.sum()
    N = 6
    for step in range(1, N + 1):
        x_prev, v_prev = x, v
        x, v = orc.step(x, v, F, td, 3)
        # exact after every iteration: sum m d = h sum m v + h^2 sum F  (1^T L = 0)
        lhs = (m[:, None] * (x - x_prev)).sum(0)
        rhs = H * (m[:, None] * orc.pbd_damping(x_prev, v_prev, m, kappa)).sum(0) + H ** 2 * F.sum(0)
        assert np.allclose(lhs, rhs, rtol=1e-10, atol=1e-14)
        cm = (m[:, None] * x).sum(0) / m.sum()
        closed = H ** 2 * F.sum(0) / m.sum() * step * (step + 1) / 2
        assert np.allclose(cm - cm0, closed, rtol=1e-9, atol=1e-15)


# ---- P5 ------------------------------------------------------------------------------
def test_p5_zero_stiffness_reduces_to_free_particles(ico):
    ct, _ = ico
    mat = Material(skalak_B=0.0, skalak_C=0.0, skalak_D=0.0, k_bending=0.0, k_volume=0.0,
                   rayleigh_alpha=0.0, rayleigh_beta=0.0, kappa_damping=0.0)
    td = orc.system_matrices(orc.rest_data(ct.rest_positions, ct.triangles, mat), H)
    rng = np.random.default_rng(2)
    x = ct.rest_positions + 0.1 * rng.standard_normal((12, 3))
    v = rng.standard_normal((12, 3))
    F = rng.standard_normal((12, 3))
    x1, v1 = orc.step(x, v, F, td, 1)
    expect = H * v + H ** 2 * F / td.mass[:, None]
    assert np.allclose(x1 - x, expect, rtol=1e-13, atol=1e-16)
    assert np.allclose(v1, expect / H, rtol=1e-13)


# ---- P6 ------------------------------------------------------------------------------
def test_p6_quadratic_energy_one_iteration_is_the_dense_solve(rbc162, monkeypatch):
    ct, td0 = rbc162
    td = copy.copy(td0)
    td.kappa = 0.0
    monkeypatch.setattr(orc, "grad_energy", lambda x, t: np.einsum("ij,...jc->...ic", t.L, x))
    rng = np.random.default_rng(9)
    x = ct.rest_positions + 0.02 * rng.standard_normal(ct.rest_positions.shape)
    v = 0.1 * rng.standard_normal(x.shape)
    F = rng.standard_normal(x.shape)
    x1, _ = orc.step(x, v, F, td, 1)
    M = np.diag(td.mass)
    A = td.M_tilde / H ** 2 + td.L
    rhs = td.M_tilde @ x / H ** 2 + M @ v / H + F           # stationarity of Eq. (3), E = x^T L x / 2
    x_ref = np.linalg.solve(A, rhs)
    assert np.allclose(x1, x_ref, rtol=1e-11, atol=1e-12)
    x2, _ = orc.step(x, v, F, td, 2)                        # a second iteration changes nothing
    assert np.allclose(x2, x1, rtol=1e-11, atol=1e-12)


# ---- P7 ------------------------------------------------------------------------------
def test_p7_converged_step_satisfies_newton_second_law(ico):
    ct, td = ico
    rng = np.random.default_rng(4)
    x = ct.rest_positions + 0.05 * rng.standard_normal((12, 3))
    v = 0.05 * rng.standard_normal((12, 3))
    F = 5.0 * rng.standard_normal((12, 3))
    x1, v1, hist = orc.step(x, v, F, td, 400, record=True)
    res = orc.eq2_residual(hist["v_damped"], x1, v1, F, td)
    assert np.abs(res).max() < 1e-9 * np.abs(F).max()
    # and far from converged after one iteration: the test is not vacuous
    xa, va, ha = orc.step(x, v, F, td, 1, record=True)
    assert np.abs(orc.eq2_residual(ha["v_damped"], xa, va, F, td)).max() > 1e-4


def _rayleigh_type(ct, alpha, beta, kappa=0.0):
    import dataclasses
    mat = dataclasses.replace(ct.material, rayleigh_alpha=alpha, rayleigh_beta=beta, kappa_damping=kappa)
    return dataclasses.replace(ct, material=mat)


def test_p6_p7_rayleigh_alpha_nonzero_system_matrices(rbc162, ico, monkeypatch):
    """The alpha_D != 0 branch of `system_matrices` (PAPER.md:234 lists alpha_D = 0, but PAPER.md:264 defines
    C = alpha_D M + beta_D K as part of the model): M~ = M + h C = (1 + h alpha) M + h beta L, written out HERE from
    M, L_cot, alpha, beta, h - not taken from the oracle's M~.  A dropped or mis-scaled alpha term (e.g. M~ = M +
    h beta L, or alpha M without the factor h) fails both parts."""
    alpha, beta = 0.3, 0.01                                    # 1/us, us
    # ---- P6 with alpha: one iteration on a purely quadratic energy equals the dense solve ----------
    ct, _ = rbc162
    td = orc.make_type(_rayleigh_type(ct, alpha, beta), H)
    M = np.diag(td.rho * td.volume0 * td.area_vertex / td.area_total)
    L = (td.B + 2 * td.C) * td.L_cot + td.k_b * td.L_cot.T @ np.diag(1.0 / td.area_vertex) @ td.L_cot
    C_damp = alpha * M + beta * L
    M_tilde = M + H * C_damp
    assert np.allclose(td.M_tilde, M_tilde, rtol=1e-13, atol=0)
    assert not np.allclose(td.M_tilde, M + H * beta * L, rtol=1e-3)          # the alpha term is not negligible here
    monkeypatch.setattr(orc, "grad_energy", lambda x, t: np.einsum("ij,...jc->...ic", t.L, x))
    rng = np.random.default_rng(19)
    x = ct.rest_positions + 0.02 * rng.standard_normal(ct.rest_positions.shape)
    v = 0.1 * rng.standard_normal(x.shape)
    F = rng.standard_normal(x.shape)
    x1, _ = orc.step(x, v, F, td, 1)
    x_ref = np.linalg.solve(M_tilde / H ** 2 + L, M_tilde @ x / H ** 2 + M @ v / H + F)
    assert np.allclose(x1, x_ref, rtol=1e-11, atol=1e-12)
    monkeypatch.undo()
    # ---- P7 with alpha: the converged step satisfies Eq. (2) with C = alpha M + beta L spelled out ----
    ct, _ = ico
    td = orc.make_type(_rayleigh_type(ct, alpha, beta), H)
    M = np.diag(td.mass)
    L = (td.B + 2 * td.C) * td.L_cot + td.k_b * td.L_cot.T @ np.diag(1.0 / td.area_vertex) @ td.L_cot
    C_damp = alpha * M + beta * L
    x = ct.rest_positions + 0.05 * rng.standard_normal((12, 3))
    v = 0.05 * rng.standard_normal((12, 3))
    F = 5.0 * rng.standard_normal((12, 3))
    x1, v1, hist = orc.step(x, v, F, td, 400, record=True)
    res = M @ (v1 - hist["v_damped"]) / H - (-orc.grad_energy(x1, td) + F - C_damp @ v1)      # Eq. (2)
    assert np.abs(res).max() < 1e-9 * np.abs(F).max()
    res_no_alpha = M @ (v1 - hist["v_damped"]) / H - (-orc.grad_energy(x1, td) + F - beta * L @ v1)
    assert np.abs(res_no_alpha).max() > 1e-4 * np.abs(F).max()                # dropping alpha M v is visible


# ---- P8 ------------------------------------------------------------------------------
def test_p8_icosahedron_brute_force_minimiser(ico):
    ct, td = ico
    rng = np.random.default_rng(8)
    x = ct.rest_positions + 0.05 * rng.standard_normal((12, 3))
    v = 0.02 * rng.standard_normal((12, 3))
    F = 3.0 * rng.standard_normal((12, 3))
    x1, v1, hist = orc.step(x, v, F, td, 600, record=True)
    obj = np.array([float(o) for o in hist["objective"]])
    assert np.all(np.diff(obj) <= 1e-12 * np.abs(obj).max())       # monotone decrease in k
    vd = hist["v_damped"]
    b = td.mass[:, None] * vd / H + F

    def fun(dflat):
        return float(orc.objective(dflat.reshape(12, 3), x, b, td))

    # independent minimiser built from objective VALUES only: BFGS on finite-difference
    # gradients, polished by Newton steps with a finite-difference Hessian
    res = scipy.optimize.minimize(fun, (H * vd).ravel(), method="BFGS", jac="3-point",
                                  options={"gtol": 1e-10, "maxiter": 5000})

    def fd_grad(z, eps=1e-5):
        out = np.empty_like(z)
        for i in range(z.size):
            zp, zm = z.copy(), z.copy()
            zp[i] += eps
            zm[i] -= eps
            out[i] = (fun(zp) - fun(zm)) / (2 * eps)
        return out

    z = res.x.copy()
    for _ in range(3):
        g0 = fd_grad(z)
        hess = np.empty((z.size, z.size))
        for i in range(z.size):
            zp, zm = z.copy(), z.copy()
            zp[i] += 1e-4
            zm[i] -= 1e-4
            hess[:, i] = (fd_grad(zp) - fd_grad(zm)) / 2e-4
        z = z - np.linalg.solve(0.5 * (hess + hess.T), g0)
    res.x, res.fun = z, fun(z)
    d_ref = res.x.reshape(12, 3)
    d = x1 - x
    assert np.linalg.norm(d - d_ref) < 2e-6 * np.linalg.norm(d)
    assert fun(d.ravel()) <= res.fun + 1e-10 * abs(res.fun)


# ---- P9 ------------------------------------------------------------------------------
@pytest.mark.parametrize("s", [0.9, 1.07])
def test_p9_uniform_scaling_closed_forms(rbc162, s):
    ct, td = rbc162
    x = s * ct.rest_positions
    I1, I2, _ = orc.strain_invariants(x, td)
    assert np.allclose(I1, 2 * s ** 2 - 2, rtol=1e-12)
    assert np.allclose(I2, s ** 4 - 1, rtol=1e-11)
    e = orc.energies(x, td)
    A, V0 = td.area_total, td.volume0
    i1, i2 = 2 * s ** 2 - 2, s ** 4 - 1
    assert e["strain"] == pytest.approx(A * (td.B / 4) * (0.5 * i1 ** 2 + i1 - i2), rel=1e-11)
    assert e["area"] == pytest.approx(A * (td.C / 8) * i2 ** 2, rel=1e-11)
    assert abs(e["bend"]) < 1e-18
    assert e["volume"] == pytest.approx(0.5 * td.k_v * (s ** 3 - 1) ** 2 * V0, rel=1e-11)


# ---- P10 -----------------------------------------------------------------------------
def test_p10_icosahedron_textbook(ico):
    ct, td = ico
    R = 3.0
    a = R / math.sin(2 * math.pi / 5)                    # edge from circumradius
    assert a == pytest.approx(3.15438, abs=1e-5)
    assert td.hinge.shape == (30, 4)
    assert np.allclose(td.theta0, math.pi - math.acos(-math.sqrt(5) / 3), rtol=1e-12)
    assert td.theta0[0] == pytest.approx(0.729728, abs=1e-6)
    assert td.volume0 == pytest.approx(5 / 12 * (3 + math.sqrt(5)) * a ** 3, rel=1e-12)
    assert td.volume0 == pytest.approx(68.4761, abs=1e-4)
    assert td.area_total == pytest.approx(5 * math.sqrt(3) * a ** 2, rel=1e-12)
    assert td.area_total == pytest.approx(86.1709, abs=1e-4)
    assert np.allclose(td.area_vertex, td.area_total / 12)
    # lumped mass sums to density * volume (total mass incl. interior fluid)
    assert td.mass.sum() == pytest.approx(1025.0 * td.volume0, rel=1e-12)


# ---- P11 -----------------------------------------------------------------------------
def test_p11_cotangent_laplacian(rbc162):
    ct, td = rbc162
    X, tri = ct.rest_positions, ct.triangles
    n = X.shape[0]
    ref = np.zeros((n, n))
    for t in tri:
        for c in range(3):
            i, j, k = t[c], t[(c + 1) % 3], t[(c + 2) % 3]
            u, w = X[i] - X[k], X[j] - X[k]                 # angle at k opposite edge (i, j)
            cot = np.dot(u, w) / np.linalg.norm(np.cross(u, w))
            ref[i, j] -= 0.5 * cot
            ref[j, i] -= 0.5 * cot
            ref[i, i] += 0.5 * cot
            ref[j, j] += 0.5 * cot
    assert np.allclose(td.L_cot, ref, rtol=1e-10, atol=1e-12)
    assert np.abs(td.L_cot.sum(axis=1)).max() < 1e-11
    ev = np.linalg.eigvalsh(td.L_cot)
    assert abs(ev[0]) < 1e-10 and ev[1] > 1e-3
    assert np.abs(td.L.sum(axis=1)).max() < 1e-6           # 1^T L = 0 (scaled by k_mem ~ 1e4)
    assert np.linalg.eigvalsh(td.H_tilde)[0] > 0           # H~ is SPD


# ---- P12 -----------------------------------------------------------------------------
def _golden_geometry():
    rows = {}
    with open(os.path.join(GOLDEN, "geometry_pins.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            name, level, vol, area, edge, tmin, tmax = line.split()
            rows[name] = (int(level), float(vol), float(area), float(edge), float(tmin), float(tmax))
    return rows


@pytest.mark.parametrize("name", ["RBC-642", "RBC-2562", "PLT-162"])
def test_p12_discrete_geometry(name):
    level, vol, area, edge, tmin, tmax = _golden_geometry()[name]
    ct = rbc_cell_type(level) if name.startswith("RBC") else platelet_cell_type(level)
    assert ct.name == name
    td = orc.rest_data(ct.rest_positions, ct.triangles, ct.material)
    assert td.volume0 == pytest.approx(vol, abs=6e-4)
    assert td.area_total == pytest.approx(area, abs=6e-4)
    X = ct.rest_positions
    mean_edge = np.linalg.norm(X[td.hinge[:, 0]] - X[td.hinge[:, 1]], axis=1).mean()
    assert mean_edge == pytest.approx(edge, abs=6e-4)
    if not math.isnan(tmin):
        assert td.theta0.min() == pytest.approx(tmin, abs=6e-4)
        assert td.theta0.max() == pytest.approx(tmax, abs=6e-4)


def test_p12_continuum_limits():
    # Evans-Fung continuum volume/area by quadrature (independent of the mesh code)
    R0, c0, c1, c2 = 3.91, 0.207161, 2.002558, -1.122762
    z = lambda r: 0.5 * R0 * np.sqrt(max(1 - (r / R0) ** 2, 0.0)) * (  # noqa: E731
        c0 + c1 * (r / R0) ** 2 + c2 * (r / R0) ** 4)
    vol = scipy.integrate.quad(lambda r: 2 * z(r) * 2 * np.pi * r, 0, R0)[0]
    assert vol == pytest.approx(94.09, abs=0.02)
    vols = [orc.rest_data(*(lambda c: (c.rest_positions, c.triangles, c.material))(rbc_cell_type(l))).volume0
            for l in (2, 3, 4)]
    assert vols[0] < vols[1] < vols[2] < vol
    assert vol - vols[2] < 0.25 * (vol - vols[1]) * 1.2    # second-order convergence to the continuum
    plt = platelet_cell_type(4)
    assert orc.rest_data(plt.rest_positions, plt.triangles, plt.material).volume0 == pytest.approx(
        4 / 3 * math.pi * 1.8 * 1.8 * 0.5, rel=3e-3)


# ---- P13 -----------------------------------------------------------------------------
def test_p13_pbd_damping_invariants(rbc162):
    ct, td = rbc162
    rng = np.random.default_rng(6)
    x = ct.rest_positions + rng.uniform(-30, 30, 3)
    v = rng.standard_normal(x.shape)
    m = td.mass
    cm = (m[:, None] * x).sum(0) / m.sum()
    for kappa in (0.3, 0.5, 1.0):
        vd = orc.pbd_damping(x, v, m, kappa)
        assert np.allclose((m[:, None] * vd).sum(0), (m[:, None] * v).sum(0), rtol=1e-12)
        assert np.allclose(np.cross(x - cm, m[:, None] * vd).sum(0),
                           np.cross(x - cm, m[:, None] * v).sum(0), rtol=1e-10)
    # kappa = 1 leaves a rigid velocity field, and a rigid field is a fixed point for any kappa
    v_rigid = orc.pbd_damping(x, v, m, 1.0)
    w = np.linalg.lstsq(np.concatenate([np.cross(np.eye(3)[i], x - cm) for i in range(3)]).reshape(3, -1).T,
                        (v_rigid - (m[:, None] * v).sum(0) / m.sum()).ravel(), rcond=None)
    assert w[1].size == 0 or w[1][0] < 1e-18
    assert np.allclose(orc.pbd_damping(x, v_rigid, m, 0.7), v_rigid, rtol=1e-11, atol=1e-13)
    # kappa = 0 is the identity
    assert np.array_equal(orc.pbd_damping(x, v, m, 0.0), v)


# ---- batching ------------------------------------------------------------------------
def test_batched_cells_equal_one_by_one(rbc162):
    ct, td = rbc162
    rng = np.random.default_rng(10)
    x = ct.rest_positions[None] + 0.02 * rng.standard_normal((4,) + ct.rest_positions.shape)
    v = 0.05 * rng.standard_normal(x.shape)
    F = rng.standard_normal(x.shape)
    xb, vb = orc.step(x, v, F, td, 4)
    for c in range(4):
        xc, vc = orc.step(x[c], v[c], F[c], td, 4)
        assert np.allclose(xb[c], xc, rtol=1e-13, atol=1e-14)
        assert np.allclose(vb[c], vc, rtol=1e-11, atol=1e-13)


def test_mesh_counts():
    for level in range(0, 4):
        v, f = icosphere(level)
        assert v.shape[0] == 10 * 4 ** level + 2 and f.shape[0] == 20 * 4 ** level
        hinges = orc.build_hinges(f.astype(np.int64))
        assert hinges.shape[0] == 30 * 4 ** level
        valence = np.bincount(hinges[:, :2].ravel(), minlength=v.shape[0])
        assert np.sum(valence == 5) == 12 and np.all((valence == 5) | (valence == 6))
        # outward orientation: positive enclosed volume
        assert orc.enclosed_volume(v, f.astype(np.int64)) > 0


# ---- Armijo line search + gradient-norm stopping test (oracle.step_line_search) ----
def _violent_case():
    """RBC-162, h = 30 us, N(0, 3000 pN) forces: the plain iteration of Eq. (4) blows up (SURVEY.md
    section 4: 'unconditional stability ... only holds with a line search')."""
    import warnings
    from workloads.meshes import rbc_cell_type
    ct = rbc_cell_type(2)
    td = orc.make_type(ct, 30.0)
    rng = np.random.default_rng(0)
    x = np.repeat(ct.rest_positions[None], 2, axis=0)
    f = 3000.0 * rng.standard_normal(x.shape)
    warnings.filterwarnings("ignore")
    return td, x, np.zeros_like(x), f


def test_ls_accepts_full_steps_where_the_plain_iteration_descends(rbc162):
    ct, td = rbc162
    rng = np.random.default_rng(3)
    x = np.repeat(ct.rest_positions[None], 3, axis=0)
    f = rng.standard_normal(x.shape)
    xa, va = orc.step(x, 0 * x, f, td, 8)
    xb, vb, hist = orc.step_line_search(x, 0 * x, f, td, 8, record=True)
    assert all(np.all(a == 1.0) for a in hist["alpha"])
    assert np.array_equal(xa, xb) and np.array_equal(va, vb)


def test_ls_keeps_the_objective_monotone_where_the_plain_iteration_blows_up():
    td, x, v, f = _violent_case()
    try:
        xa, _, hist_plain = orc.step(x, v, f, td, 15, record=True)
        obj = np.array(hist_plain["objective"])
        plain_ok = np.all(np.isfinite(xa)) and np.all(np.diff(obj, axis=0) <= 0)
    except ValueError:                      # LAPACK refuses the NaNs of the diverged iterate
        plain_ok = False
    assert not plain_ok
    xb, vb, hist = orc.step_line_search(x, v, f, td, 15, max_halvings=8, c1=1e-4, record=True)
    obj = np.array(hist["objective"])       # [16, cells]
    assert np.all(np.isfinite(xb)) and np.all(np.diff(obj, axis=0) <= 0)
    alpha = np.array(hist["alpha"])
    assert alpha.min() < 1.0                                          # the search really backtracked
    assert np.all(np.isin(alpha, 0.5 ** np.arange(0, 9)))             # powers of 1/2 only
    assert np.all(obj[1:][alpha > 0.5 ** 8] < obj[:-1][alpha > 0.5 ** 8])
    # The Armijo inequality itself, re-evaluated here from the recorded iterate d, direction p and slope (a search
    # that ignored c1 alpha slope, or took the slope with the wrong sign, passes plain monotonicity but not this):
    # at every accepted step that did not exhaust the halvings  g(d + alpha p) <= g(d) + c1 alpha slope with
    # slope < 0, and the step length tried just before, 2 alpha, VIOLATED it (alpha is the first that passes).
    c1 = 1e-4
    slope = np.array(hist["slope"])
    assert np.all(slope < 0.0)                                        # H~ is SPD: p is a descent direction
    n_checked = n_rejected = 0
    for k in range(15):
        d, p, b = hist["d"][k], hist["p"][k], hist["b"]
        g0 = orc.objective(d, x, b, td)
        assert np.array_equal(g0, obj[k])
        for cell in range(x.shape[0]):
            a = alpha[k, cell]
            if a <= 0.5 ** 8:
                continue                                              # exhausted: taken without passing the test
            at = lambda s: orc.objective((d + s * p)[cell], x[cell], b[cell], td)   # noqa: E731
            assert at(a) <= g0[cell] + c1 * a * slope[k, cell]
            assert at(a) == obj[k + 1, cell]                          # the accepted point is the next iterate
            n_checked += 1
            if a < 1.0:
                assert at(2 * a) > g0[cell] + c1 * 2 * a * slope[k, cell]
                n_rejected += 1
    assert n_checked > 10 and n_rejected > 3                          # not vacuous


def test_ls_gradient_tolerance_freezes_converged_cells(rbc162):
    ct, td = rbc162
    rng = np.random.default_rng(4)
    x = np.repeat(ct.rest_positions[None], 2, axis=0)
    v = 1e-3 * rng.standard_normal(x.shape)
    f = rng.standard_normal(x.shape)
    # huge tolerance: every cell is "converged" at once -> d stays at its start h v (damped)
    xa, va, hist = orc.step_line_search(x, v, f, td, 5, grad_tol=1e9, record=True)
    vd = orc.pbd_damping(x, v, td.mass, td.kappa)
    assert np.all(np.array(hist["alpha"]) == 0.0)
    assert np.allclose(xa, x + td.h * vd, rtol=0, atol=1e-15) and np.allclose(va, vd, rtol=0, atol=1e-15)
    # tight tolerance: cells stop once the gradient is small, and the result equals the full run to that level
    xb, _, hist_b = orc.step_line_search(x, v, f, td, 60, grad_tol=1e-6, record=True)
    xc, _ = orc.step(x, v, f, td, 60)
    alpha = np.array(hist_b["alpha"])
    assert np.all(alpha[-1] == 0.0) and np.all(alpha[0] == 1.0)       # they did stop, after working
    assert np.linalg.norm(xb - xc) <= 1e-5 * np.linalg.norm(xc - x)


# ---- velocity cap and one-ring median filter of F_ext ----
def test_velocity_cap_closed_form():
    rng = np.random.default_rng(0)
    v = rng.standard_normal((4, 50, 3)) * np.array([0.01, 0.1, 1.0, 10.0])[:, None, None]
    out = orc.cap_velocity(v, 0.5)
    speed_in, speed_out = np.linalg.norm(v, axis=-1), np.linalg.norm(out, axis=-1)
    assert np.all(speed_out <= 0.5 * (1 + 1e-15))
    slow = speed_in <= 0.5
    assert np.array_equal(out[slow], v[slow])                              # untouched below the threshold
    assert np.allclose(speed_out[~slow], 0.5, rtol=1e-14)                  # exactly on it above
    assert np.allclose(np.cross(out, v), 0.0, atol=1e-12)                  # direction kept
    assert np.array_equal(orc.cap_velocity(np.zeros((2, 3, 3)), 0.5), np.zeros((2, 3, 3)))   # no 0/0


def test_median_filter_removes_a_spike_and_keeps_a_constant(ico):
    ct, td = ico                                  # icosahedron: every vertex has exactly 5 neighbours
    ring = orc.one_ring(td.tri, td.n)
    assert all(len(r) == 5 for r in ring) and all(v not in r for v, r in enumerate(ring))
    f = np.tile(np.array([1.0, -2.0, 3.0]), (td.n, 1))
    assert np.array_equal(orc.median_filter_forces(f, td), f)              # constant field is a fixed point
    spike = f.copy()
    spike[7] = [1e6, 1e6, 1e6]
    assert np.array_equal(orc.median_filter_forces(spike, td), f)          # one outlier never reaches a median of 6
    # brute force against the definition on random data (6 values: mean of the two central ones)
    rng = np.random.default_rng(1)
    g = rng.standard_normal((3, td.n, 3))
    out = orc.median_filter_forces(g, td)
    for c in range(3):
        for v in range(td.n):
            for k in range(3):
                vals = sorted([g[c, v, k]] + [g[c, u, k] for u in ring[v]])
                assert out[c, v, k] == 0.5 * (vals[2] + vals[3])


def test_median_filter_odd_count_brute_force(rbc162):
    """Valence-6 vertices: 7 values per median (the vertex + 6 neighbours), the ODD-count branch of reading R18 -
    the icosahedron above only has even counts.  Brute force against the definition: the 4th of the 7 sorted values;
    the 12 valence-5 vertices of the icosphere (6 values) average the two central ones."""
    ct, td = rbc162
    ring = orc.one_ring(td.tri, td.n)
    counts = np.array([len(r) for r in ring])
    assert set(counts) == {5, 6} and np.sum(counts == 5) == 12
    rng = np.random.default_rng(2)
    g = rng.standard_normal((2, td.n, 3))
    out = orc.median_filter_forces(g, td)
    for c in range(2):
        for v in range(td.n):
            for k in range(3):
                vals = sorted([g[c, v, k]] + [g[c, u, k] for u in ring[v]])
                expect = vals[3] if len(vals) == 7 else 0.5 * (vals[2] + vals[3])
                assert out[c, v, k] == expect
    # a spike is removed at an odd count too, and lands in no neighbour's median
    f = np.tile(np.array([1.0, -2.0, 3.0]), (td.n, 1))
    spike = f.copy()
    v6 = int(np.nonzero(counts == 6)[0][0])
    spike[v6] = 1e6
    assert np.array_equal(orc.median_filter_forces(spike, td), f)


def test_step_with_cap_only_changes_the_velocity(rbc162):
    ct, td = rbc162
    rng = np.random.default_rng(5)
    x = ct.rest_positions[None]
    f = 50.0 * rng.standard_normal(x.shape)
    xa, va = orc.step(x, 0 * x, f, td, 4)
    xb, vb = orc.step(x, 0 * x, f, td, 4, v_max=1e-4)
    assert np.array_equal(xa, xb) and np.linalg.norm(va, axis=-1).max() > 1e-4
    assert np.array_equal(vb, orc.cap_velocity(va, 1e-4))


# ---- PIK collision energy ----
def test_collision_energy_closed_forms_and_gradient(rbc162):
    ct, td = rbc162
    rng = np.random.default_rng(6)
    x = ct.rest_positions + 0.05 * rng.standard_normal(ct.rest_positions.shape)
    k = np.where(rng.random(td.n) < 0.3, rng.uniform(10, 200, td.n), 0.0)       # 30 % of the vertices in contact
    t = np.array([0.3, -0.2, 0.1])
    # rigid offset from the targets: E = 1/2 sum k |t|^2, gradient k t; zero at the targets
    assert np.isclose(orc.collision_energy(x + t, x, k), 0.5 * k.sum() * t @ t, rtol=1e-14)
    assert np.allclose(orc.grad_collision(x + t, x, k), k[:, None] * t, rtol=1e-14)
    assert orc.collision_energy(x, x, k) == 0.0 and not orc.grad_collision(x, x, k).any()
    # central finite differences of the energy against the analytic gradient
    p = x + 0.1 * rng.standard_normal(x.shape)
    g = orc.grad_collision(x, p, k)
    for v, c in [(0, 0), (5, 1), (17, 2), (100, 0)]:
        e = np.zeros_like(x); e[v, c] = 1e-6
        fd = (orc.collision_energy(x + e, p, k) - orc.collision_energy(x - e, p, k)) / 2e-6
        assert np.isclose(fd, g[v, c], rtol=1e-7, atol=1e-9)


def test_step_with_collisions_pulls_flagged_vertices_to_their_targets(rbc162):
    ct, td = rbc162
    x = ct.rest_positions[None]
    k = np.zeros((1, td.n)); flagged = [3, 40, 41, 90]; k[0, flagged] = 400.0
    targets = x + np.array([0.0, 0.0, 0.02])                      # push the flagged vertices 20 nm up
    f = np.zeros_like(x)
    xa, _ = orc.step(x, 0 * x, f, td, 10)                          # rest state: nothing moves (pin P1)
    assert np.abs(xa - x).max() < 1e-10
    xb, _, hist = orc.step(x, 0 * x, f, td, 40, collisions=(targets, k), record=True)
    obj = np.array(hist["objective"])[:, 0]
    assert np.all(np.diff(obj) <= 1e-12 * np.abs(obj[:-1]).max())  # the constant-H~ iteration still descends (R19)
    moved = (xb - x)[0, :, 2]
    assert np.all(moved[flagged] > 1e-4) and moved[flagged].min() > 5 * np.abs(np.delete(moved, flagged)).mean()
    # k = 0 everywhere is exactly the plain step
    xc, _ = orc.step(x, 0 * x, f, td, 10, collisions=(targets, 0 * k))
    assert np.array_equal(xc, xa)


def test_reduced_gradient_form_of_the_iteration(rbc162):
    """The identity the fast GPU kernels are built on, checked on the ORACLE's matrices:
    with H~ = M~/h^2 + L, M~ = (1 + h alpha) M + h beta L and gamma = (beta/h) / (1 + beta/h),
        M~/h^2 = (1 - gamma) m^ + gamma H~,      m^ = (1 + h alpha) M / h^2,
    so grad g = r + gamma H~ d with the reduced gradient r = (1 - gamma) m^ d - b + grad E, and Eq. (4)
    d <- d - H~^-1 grad g is exactly d <- (1 - gamma) d - H~^-1 r.  The line search's damping kernel adds
    gamma m^ d + (beta/h) L d to r, which is the same full gradient."""
    ct, td = rbc162
    assert td.beta > 0.0
    rng = np.random.default_rng(3)
    n = td.mass.shape[0]
    d = 0.01 * rng.standard_normal((n, 3))
    b = rng.standard_normal((n, 3))
    x_n = ct.rest_positions + 0.02 * rng.standard_normal((n, 3))
    gamma = (td.beta / td.h) / (1.0 + td.beta / td.h)
    m_hat = (1.0 + td.h * td.alpha) * td.mass[:, None] / td.h ** 2
    assert np.allclose(td.M_tilde / td.h ** 2, (1.0 - gamma) * np.diag(m_hat[:, 0]) + gamma * td.H_tilde,
                       rtol=1e-12, atol=1e-12 * np.abs(td.H_tilde).max())
    full = orc.gradient_g(d, x_n, b, td)
    r = (1.0 - gamma) * m_hat * d - b + orc.grad_energy(x_n + d, td)
    scale = np.abs(full).max()
    assert np.abs(r + gamma * (td.H_tilde @ d) - full).max() <= 1e-12 * scale
    assert np.abs(r + gamma * m_hat * d + (td.beta / td.h) * (td.L @ d) - full).max() <= 1e-12 * scale
    plain = d - orc.solve_H_tilde(full, td)
    reduced = (1.0 - gamma) * d - orc.solve_H_tilde(r, td)
    assert np.abs(plain - reduced).max() <= 1e-10 * np.abs(plain).max()
