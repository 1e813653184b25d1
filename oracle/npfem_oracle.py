"""fp64 CPU oracle for the npFEM solid-solver step.  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import this module.  It shares no code with the
CUDA path (`paper_1911_03062_b200/`) and imports nothing from it.

What it follows (citations are /root/reference/PAPER.md lines):
  * Eqs. (1)-(2), implicit Euler advancement ................. PAPER.md:257-264
  * Eq. (3), variational form, M~ = M + hC, y_n .............. PAPER.md:266-268
  * Eq. (4), quasi-Newton iteration with a constant H~ ....... PAPER.md:268-272
  * material constants ....................................... PAPER.md:226-239
  * lumped mass, Rayleigh + position-based-dynamics damping .. PAPER.md:264
The paper defers the energies, H~ and the damping formulas to its ref. [4]
(not available); every gap is filled by the readings R1-R16 of SURVEY.md
section 8(c), restated in DESIGN.md.  It is an ITERATION (fixed K), so the
oracle is the algorithm step by step in the paper's order; the only library
primitive used as a step is LAPACK's Cholesky factor/solve (scipy.linalg).

Pins: tests/test_oracle_pins.py (P1-P13 of SURVEY.md section 8(c)).
PARITY UNPINNED for: the line-search constants of `step_line_search` (Armijo c1, halving factor 1/2:
conventional choices, the paper has no line search), the unused Skalak constant D (R6), the platelet stiffness
factor (R13), and fidelity to the authors' actual npFEM energies - parity with
the published npFEM is not claimed.

All arrays are float64; every function accepts a leading batch of cells:
positions x have shape [..., n, 3] (the paper's x in R^{n x 3}).
Units: um, us, fg, pN.
"""
from __future__ import annotations

import dataclasses

import numpy as np
import scipy.linalg


# --------------------------------------------------------------------------------------
# rest data of one cell type
# --------------------------------------------------------------------------------------
@dataclasses.dataclass
class TypeData:
    n: int
    tri: np.ndarray          # [T,3]
    hinge: np.ndarray        # [E,4] columns i, j, k, l
    dm_a: np.ndarray         # [T] Dm^-1 = [[a, b], [0, c]]
    dm_b: np.ndarray
    dm_c: np.ndarray
    area0: np.ndarray        # [T] rest triangle areas
    theta0: np.ndarray       # [E] rest hinge angles
    volume0: float
    area_total: float
    area_vertex: np.ndarray  # [n]
    # material
    B: float
    C: float
    k_b: float
    k_v: float
    alpha: float
    beta: float
    kappa: float
    rho: float
    # constant matrices for time step h
    h: float = 0.0
    mass: np.ndarray = None      # [n]   lumped M
    L_cot: np.ndarray = None     # [n,n]
    L: np.ndarray = None         # [n,n]
    M_tilde: np.ndarray = None   # [n,n] = M + hC
    H_tilde: np.ndarray = None   # [n,n] = M~/h^2 + L
    H_chol: tuple = None         # scipy cho_factor of H~


def build_hinges(tri: np.ndarray) -> np.ndarray:
    """All edges of a closed oriented 2-manifold as hinges (i, j, k, l), i < j.

    k = vertex opposite the directed edge i->j in the triangle that contains it,
    l = opposite vertex of the other triangle.
    """
    opposite: dict[tuple[int, int], int] = {}
    for a, b, c in tri.tolist():
        for u, v, w in ((a, b, c), (b, c, a), (c, a, b)):
            if (u, v) in opposite:
                raise ValueError("directed edge appears twice: surface not oriented/manifold")
            opposite[(u, v)] = w
    hinges = []
    for (u, v), w in opposite.items():
        if (v, u) not in opposite:
            raise ValueError("edge without a twin: surface not closed")
        if u < v:
            hinges.append((u, v, w, opposite[(v, u)]))
    hinges.sort()
    return np.array(hinges, dtype=np.int64).reshape(-1, 4)


def hinge_angles(x: np.ndarray, hinge: np.ndarray) -> np.ndarray:
    """theta = atan2((n_A x n_B).e^, n_A.n_B), n_A = e x (x_k - x_i), n_B = (x_l - x_i) x e."""
    xi, xj = x[..., hinge[:, 0], :], x[..., hinge[:, 1], :]
    xk, xl = x[..., hinge[:, 2], :], x[..., hinge[:, 3], :]
    e = xj - xi
    n_a = np.cross(e, xk - xi)
    n_b = np.cross(xl - xi, e)
    e_hat = e / np.linalg.norm(e, axis=-1, keepdims=True)
    sin_part = np.sum(np.cross(n_a, n_b) * e_hat, axis=-1)
    cos_part = np.sum(n_a * n_b, axis=-1)
    return np.arctan2(sin_part, cos_part)


def enclosed_volume(x: np.ndarray, tri: np.ndarray) -> np.ndarray:
    """V = sum_t x0 . (x1 x x2) / 6."""
    x0, x1, x2 = x[..., tri[:, 0], :], x[..., tri[:, 1], :], x[..., tri[:, 2], :]
    return np.sum(np.sum(x0 * np.cross(x1, x2), axis=-1), axis=-1) / 6.0


def rest_data(rest_positions: np.ndarray, triangles: np.ndarray, material) -> TypeData:
    """Per-type rest quantities (SURVEY.md 8(c) 'Per cell type, once')."""
    X = np.asarray(rest_positions, dtype=np.float64)
    tri = np.asarray(triangles, dtype=np.int64)
    n = X.shape[0]
    E1 = X[tri[:, 1]] - X[tri[:, 0]]
    E2 = X[tri[:, 2]] - X[tri[:, 0]]
    len1 = np.linalg.norm(E1, axis=1)
    E1_hat = E1 / len1[:, None]
    proj = np.sum(E2 * E1_hat, axis=1)
    height = np.linalg.norm(E2 - proj[:, None] * E1_hat, axis=1)
    # Dm = [[len1, proj], [0, height]]  ->  Dm^-1 = [[1/len1, -proj/(len1*height)], [0, 1/height]]
    dm_a = 1.0 / len1
    dm_b = -proj / (len1 * height)
    dm_c = 1.0 / height
    area0 = 0.5 * len1 * height
    area_vertex = np.zeros(n)
    for c in range(3):
        np.add.at(area_vertex, tri[:, c], area0 / 3.0)
    hinge = build_hinges(tri)
    return TypeData(
        n=n, tri=tri, hinge=hinge, dm_a=dm_a, dm_b=dm_b, dm_c=dm_c, area0=area0,
        theta0=hinge_angles(X, hinge), volume0=float(enclosed_volume(X, tri)),
        area_total=float(np.sum(area0)), area_vertex=area_vertex,
        B=float(material.skalak_B), C=float(material.skalak_C),
        k_b=float(material.k_bending), k_v=float(material.k_volume),
        alpha=float(material.rayleigh_alpha), beta=float(material.rayleigh_beta),
        kappa=float(material.kappa_damping), rho=float(material.density))


# --------------------------------------------------------------------------------------
# constant matrices (reading R4, R10, R11 of SURVEY.md 8(c))
# --------------------------------------------------------------------------------------
def cotangent_matrix(td: TypeData) -> np.ndarray:
    """L_cot = sum_t A0_t G_t G_t^T, G_t = [[-1,-1],[1,0],[0,1]] Dm_t^-1 (3x2)."""
    L = np.zeros((td.n, td.n))
    for t in range(td.tri.shape[0]):
        a, b, c = td.dm_a[t], td.dm_b[t], td.dm_c[t]
        dm_inv = np.array([[a, b], [0.0, c]])
        G = np.array([[-1.0, -1.0], [1.0, 0.0], [0.0, 1.0]]) @ dm_inv
        idx = td.tri[t]
        L[np.ix_(idx, idx)] += td.area0[t] * (G @ G.T)
    return L


def system_matrices(td: TypeData, h: float) -> TypeData:
    """M (lumped), L, M~ = M + hC with C = alpha M + beta L, H~ = M~/h^2 + L; Cholesky of H~."""
    td.h = float(h)
    td.L_cot = cotangent_matrix(td)
    k_mem = td.B + 2.0 * td.C
    td.L = k_mem * td.L_cot + td.k_b * td.L_cot.T @ np.diag(1.0 / td.area_vertex) @ td.L_cot
    td.mass = td.rho * td.volume0 * td.area_vertex / td.area_total          # R10
    td.M_tilde = (1.0 + h * td.alpha) * np.diag(td.mass) + h * td.beta * td.L
    td.H_tilde = td.M_tilde / h ** 2 + td.L
    td.H_chol = scipy.linalg.cho_factor(td.H_tilde, lower=True)
    return td


def make_type(cell_type, h: float) -> TypeData:
    """Convenience: rest data + matrices from a workloads.CellType-like object."""
    td = rest_data(cell_type.rest_positions, cell_type.triangles, cell_type.material)
    return system_matrices(td, h)


# --------------------------------------------------------------------------------------
# energies  E = E_strain + E_area + E_bend + E_vol   (F_int = -grad E)
# --------------------------------------------------------------------------------------
def strain_invariants(x: np.ndarray, td: TypeData):
    """Per triangle: F = [e1 e2] Dm^-1, C = F^T F, I1 = tr C - 2, I2 = det C - 1."""
    tri = td.tri
    e1 = x[..., tri[:, 1], :] - x[..., tri[:, 0], :]
    e2 = x[..., tri[:, 2], :] - x[..., tri[:, 0], :]
    f1 = td.dm_a[:, None] * e1
    f2 = td.dm_b[:, None] * e1 + td.dm_c[:, None] * e2
    C11 = np.sum(f1 * f1, axis=-1)
    C12 = np.sum(f1 * f2, axis=-1)
    C22 = np.sum(f2 * f2, axis=-1)
    I1 = C11 + C22 - 2.0
    I2 = C11 * C22 - C12 * C12 - 1.0
    return I1, I2, (f1, f2, C11, C12, C22)


def energies(x: np.ndarray, td: TypeData) -> dict:
    """The four energy families, each summed over its elements; values per cell."""
    I1, I2, _ = strain_invariants(x, td)
    e_strain = np.sum(td.area0 * (td.B / 4.0) * (0.5 * I1 ** 2 + I1 - I2), axis=-1)
    e_area = np.sum(td.area0 * (td.C / 8.0) * I2 ** 2, axis=-1)
    theta = hinge_angles(x, td.hinge)
    e_bend = np.sum(td.k_b * (1.0 - np.cos(theta - td.theta0)), axis=-1)
    vol = enclosed_volume(x, td.tri)
    e_vol = 0.5 * td.k_v * (vol - td.volume0) ** 2 / td.volume0
    return {"strain": e_strain, "area": e_area, "bend": e_bend, "volume": e_vol}


def total_energy(x: np.ndarray, td: TypeData) -> np.ndarray:
    e = energies(x, td)
    return e["strain"] + e["area"] + e["bend"] + e["volume"]


def _scatter_add(out: np.ndarray, index: np.ndarray, values: np.ndarray) -> None:
    """out[..., index[e], :] += values[..., e, :] for every element e."""
    np.add.at(out, (Ellipsis, index, slice(None)), values)


def grad_membrane(x: np.ndarray, td: TypeData) -> np.ndarray:
    """Gradient of E_strain + E_area (two-invariant Skalak law, reading R5/R7)."""
    _, I2, (f1, f2, C11, C12, C22) = strain_invariants(x, td)
    I1 = C11 + C22 - 2.0
    W1 = (td.B / 4.0) * (I1 + 1.0)                    # dW/dI1
    W2 = -td.B / 4.0 + (td.C / 4.0) * I2              # dW/dI2
    # S = 2 (W1 Id + W2 adj C),  adj C = [[C22, -C12], [-C12, C11]]
    S11 = 2.0 * (W1 + W2 * C22)
    S12 = -2.0 * W2 * C12
    S22 = 2.0 * (W1 + W2 * C11)
    P1 = S11[..., None] * f1 + S12[..., None] * f2    # P = F S, columns P1, P2
    P2 = S12[..., None] * f1 + S22[..., None] * f2
    # [dE/dx1 dE/dx2] = A0 P Dm^-T,  Dm^-T = [[a, 0], [b, c]]
    a, b, c, A0 = td.dm_a[:, None], td.dm_b[:, None], td.dm_c[:, None], td.area0[:, None]
    g1 = A0 * (a * P1 + b * P2)
    g2 = A0 * (c * P2)
    g0 = -(g1 + g2)
    out = np.zeros_like(x)
    _scatter_add(out, td.tri[:, 0], g0)
    _scatter_add(out, td.tri[:, 1], g1)
    _scatter_add(out, td.tri[:, 2], g2)
    return out


def grad_bending(x: np.ndarray, td: TypeData) -> np.ndarray:
    """Gradient of E_bend = k_b (1 - cos(theta - theta0)) per hinge (reading R8)."""
    hg = td.hinge
    xi, xj = x[..., hg[:, 0], :], x[..., hg[:, 1], :]
    xk, xl = x[..., hg[:, 2], :], x[..., hg[:, 3], :]
    e = xj - xi
    n_a = np.cross(e, xk - xi)
    n_b = np.cross(xl - xi, e)
    len_e = np.linalg.norm(e, axis=-1, keepdims=True)
    na2 = np.sum(n_a * n_a, axis=-1, keepdims=True)
    nb2 = np.sum(n_b * n_b, axis=-1, keepdims=True)
    theta = hinge_angles(x, hg)
    dE = (td.k_b * np.sin(theta - td.theta0))[..., None]          # dE/dtheta
    grad_k = -len_e * n_a / na2
    grad_l = -len_e * n_b / nb2
    dot = lambda u, v: np.sum(u * v, axis=-1, keepdims=True)      # noqa: E731
    grad_i = dot(xj - xk, e) / (len_e * na2) * n_a + dot(xj - xl, e) / (len_e * nb2) * n_b
    grad_j = dot(xk - xi, e) / (len_e * na2) * n_a + dot(xl - xi, e) / (len_e * nb2) * n_b
    out = np.zeros_like(x)
    _scatter_add(out, hg[:, 0], dE * grad_i)
    _scatter_add(out, hg[:, 1], dE * grad_j)
    _scatter_add(out, hg[:, 2], dE * grad_k)
    _scatter_add(out, hg[:, 3], dE * grad_l)
    return out


def grad_volume(x: np.ndarray, td: TypeData) -> np.ndarray:
    """Gradient of E_vol = (k_v/2)(V - V0)^2 / V0 (reading R9)."""
    tri = td.tri
    x0, x1, x2 = x[..., tri[:, 0], :], x[..., tri[:, 1], :], x[..., tri[:, 2], :]
    vol = enclosed_volume(x, tri)
    coeff = (td.k_v * (vol - td.volume0) / td.volume0)[..., None, None]
    out = np.zeros_like(x)
    _scatter_add(out, tri[:, 0], np.cross(x1, x2) / 6.0)
    _scatter_add(out, tri[:, 1], np.cross(x2, x0) / 6.0)
    _scatter_add(out, tri[:, 2], np.cross(x0, x1) / 6.0)
    return coeff * out


def grad_energy(x: np.ndarray, td: TypeData) -> np.ndarray:
    """grad E(x) = -F_int(x)."""
    return grad_membrane(x, td) + grad_bending(x, td) + grad_volume(x, td)


# --------------------------------------------------------------------------------------
# time step
# --------------------------------------------------------------------------------------
def pbd_damping(x: np.ndarray, v: np.ndarray, mass: np.ndarray, kappa: float) -> np.ndarray:
    """Position-based-dynamics global velocity damping (paper's ref. [6], R12).

    v <- v + kappa (v_cm + omega x r - v),  r = x - x_cm,
    omega = I^-1 sum r x (m v),  I = sum m (|r|^2 Id - r r^T).
    """
    if kappa == 0.0:
        return v.copy()
    m = mass[:, None]
    m_tot = np.sum(mass)
    x_cm = np.sum(m * x, axis=-2, keepdims=True) / m_tot
    v_cm = np.sum(m * v, axis=-2, keepdims=True) / m_tot
    r = x - x_cm
    ang = np.sum(np.cross(r, m * v), axis=-2)                                 # [..., 3]
    r2 = np.sum(r * r, axis=-1)                                               # [..., n]
    inertia = (np.sum(mass * r2, axis=-1)[..., None, None] * np.eye(3)
               - np.einsum("v,...vi,...vj->...ij", mass, r, r))
    omega = np.linalg.solve(inertia, ang[..., None])[..., 0]
    dv = v_cm + np.cross(omega[..., None, :], r) - v
    return v + kappa * dv


def cap_velocity(v: np.ndarray, v_max: float) -> np.ndarray:
    """Vertex-velocity cap (the npFEM vertex velocity, "if it exceeds a value of U*_max,
    is truncated towards this threshold").  Reading R17: the MAGNITUDE of each vertex velocity is
    clamped to v_max, its direction kept; applied to v_{n+1} as stored."""
    speed = np.sqrt(np.sum(v * v, axis=-1, keepdims=True))
    return v * np.minimum(1.0, v_max / np.maximum(speed, np.finfo(np.float64).tiny))


def one_ring(tri: np.ndarray, n: int) -> list:
    """Sorted one-ring neighbour indices of every vertex."""
    ring = [set() for _ in range(n)]
    for a, b, c in tri:
        ring[a].update((b, c)); ring[b].update((a, c)); ring[c].update((a, b))
    return [np.array(sorted(r), dtype=np.int64) for r in ring]


def median_filter_forces(f: np.ndarray, td: TypeData) -> np.ndarray:
    """Median filter of F_ext "in the one-ring neighbourhood of every Lagrangian point".
    Reading R18: per vertex and per Cartesian component, the median over the vertex itself and its
    one-ring neighbours (an even count averages the two central values), SURVEY.md 8(f)-2."""
    out = np.empty_like(f)
    for v, ring in enumerate(one_ring(td.tri, td.n)):
        idx = np.concatenate(([v], ring))
        out[..., v, :] = np.median(f[..., idx, :], axis=-2)
    return out


def apply_M_tilde(d: np.ndarray, td: TypeData) -> np.ndarray:
    return np.einsum("ij,...jc->...ic", td.M_tilde, d)


def solve_H_tilde(g: np.ndarray, td: TypeData) -> np.ndarray:
    """H~^-1 g for every cell and the three coordinate columns (Cholesky solve)."""
    lead = g.shape[:-2]
    rhs = np.moveaxis(g.reshape((-1,) + g.shape[-2:]), 1, 0).reshape(td.n, -1)
    sol = scipy.linalg.cho_solve(td.H_chol, rhs)
    return np.moveaxis(sol.reshape(td.n, -1, 3), 0, 1).reshape(lead + (td.n, 3))


def collision_energy(x: np.ndarray, targets: np.ndarray, stiffness: np.ndarray) -> np.ndarray:
    """PIK collision energy (near contact "a collision force, coming from a quadratic
    potential energy", replaces the fluid force): sum_i 1/2 k_i |x_i - p_i|^2 over the flagged vertices
    (k_i = 0: not in contact), p_i the projection point handed over by the collision detection
    (reading R19: the term enters grad g but not the constant H~)."""
    return 0.5 * np.sum(stiffness * np.sum((x - targets) ** 2, axis=-1), axis=-1)


def grad_collision(x: np.ndarray, targets: np.ndarray, stiffness: np.ndarray) -> np.ndarray:
    return stiffness[..., None] * (x - targets)


def gradient_g(d: np.ndarray, x_n: np.ndarray, b: np.ndarray, td: TypeData, collisions=None) -> np.ndarray:
    """grad g = M~ (x - y_n)/h^2 + grad E(x) written with d = x - x_n:  M~ d/h^2 - b + grad E.

    b = M v_n/h + F_ext, because M~ y_n/h^2 = M~ x_n/h^2 + M v_n/h + F_ext.
    collisions = (targets, stiffness) adds the PIK term.
    """
    g = apply_M_tilde(d, td) / td.h ** 2 - b + grad_energy(x_n + d, td)
    if collisions is not None:
        g = g + grad_collision(x_n + d, *collisions)
    return g


def objective(d: np.ndarray, x_n: np.ndarray, b: np.ndarray, td: TypeData, collisions=None) -> np.ndarray:
    """g of Eq. (3) minus the d-independent constant (h^2/2) b^T M~^-1 b:

    1/(2h^2) d^T M~ d - d^T b + E(x_n + d).  Its gradient is `gradient_g`.
    """
    quad = 0.5 * np.sum(d * apply_M_tilde(d, td), axis=(-2, -1)) / td.h ** 2
    out = quad - np.sum(d * b, axis=(-2, -1)) + total_energy(x_n + d, td)
    if collisions is not None:
        out = out + collision_energy(x_n + d, *collisions)
    return out


def step(x_n: np.ndarray, v_n: np.ndarray, f_ext: np.ndarray, td: TypeData,
         n_iterations: int, record: bool = False, v_max: float = 0.0, collisions=None):
    """One time step h: {x_n, v_n} -> {x_{n+1}, v_{n+1}}.

    1. PBD damping of v_n (kappa > 0);  2. b = M v/h + F, d^0 = h v (reading R3);
    3. K times: d <- d - H~^-1 grad g (Eq. 4 with R1: the inverse; step length 1, R2);
    4. x_{n+1} = x_n + d, v_{n+1} = d/h (Eq. 1).
    """
    h = td.h
    v = pbd_damping(x_n, v_n, td.mass, td.kappa)
    b = td.mass[:, None] * v / h + f_ext
    d = h * v
    history = {"objective": [], "grad_norm": [], "v_damped": v}
    for _ in range(n_iterations):
        g = gradient_g(d, x_n, b, td, collisions)
        if record:
            history["objective"].append(objective(d, x_n, b, td, collisions))
            history["grad_norm"].append(np.sqrt(np.sum(g * g, axis=(-2, -1))))
        d = d - solve_H_tilde(g, td)
    if record:
        g = gradient_g(d, x_n, b, td, collisions)
        history["objective"].append(objective(d, x_n, b, td, collisions))
        history["grad_norm"].append(np.sqrt(np.sum(g * g, axis=(-2, -1))))
    x_next = x_n + d
    v_next = d / h
    if v_max > 0.0:
        v_next = cap_velocity(v_next, v_max)
    return (x_next, v_next, history) if record else (x_next, v_next)


def step_line_search(x_n: np.ndarray, v_n: np.ndarray, f_ext: np.ndarray, td: TypeData, n_iterations: int,
                     max_halvings: int = 8, c1: float = 1e-4, grad_tol: float = 0.0, record: bool = False):
    """`step` with a per-cell Armijo backtracking line search and a gradient-norm stopping test
    (the paper's text has neither - reading R2 - but claims "unconditional
    stability for arbitrary time steps", which the plain iteration does not have).

    Per cell and iteration k:  grad = grad g(d);  if ||grad||_2 <= grad_tol ||b||_2 the cell is
    frozen (d unchanged).  Otherwise p = -H~^-1 grad, slope = <grad, p> (< 0 because H~ is SPD),
    alpha = 1, and alpha is halved while  g(d + alpha p) > g(d) + c1 alpha slope,  at most
    `max_halvings` times (the last alpha is taken even if the test still fails).  d <- d + alpha p.
    Returns (x_next, v_next[, history]); history["alpha"] is [n_iterations] arrays of step lengths;
    history also keeps, per iteration, the slope, the iterate d and the direction p the search started from
    (and b once), so that a test can re-evaluate the Armijo inequality itself.
    """
    h = td.h
    v = pbd_damping(x_n, v_n, td.mass, td.kappa)
    b = td.mass[:, None] * v / h + f_ext
    d = h * v
    lead = d.shape[:-2]
    b_norm = np.sqrt(np.sum(b * b, axis=(-2, -1)))
    history = {"objective": [], "alpha": [], "grad_norm": [], "slope": [], "d": [], "p": [], "b": b}
    for _ in range(n_iterations):
        grad = gradient_g(d, x_n, b, td)
        g_norm = np.sqrt(np.sum(grad * grad, axis=(-2, -1)))
        frozen = g_norm <= grad_tol * b_norm
        p = -solve_H_tilde(grad, td)
        slope = np.sum(grad * p, axis=(-2, -1))
        g0 = objective(d, x_n, b, td)
        alpha = np.ones(lead)
        done = np.array(frozen, copy=True)
        for halving in range(max_halvings + 1):
            trial = objective(d + alpha[..., None, None] * p, x_n, b, td)
            ok = trial <= g0 + c1 * alpha * slope
            done = done | ok
            if halving == max_halvings or np.all(done):
                break
            alpha = np.where(done, alpha, 0.5 * alpha)
        alpha = np.where(frozen, 0.0, alpha)
        if record:
            history["slope"].append(slope)
            history["d"].append(d)
            history["p"].append(p)
        d = d + alpha[..., None, None] * p
        if record:
            history["objective"].append(g0)
            history["alpha"].append(alpha)
            history["grad_norm"].append(g_norm)
    if record:
        history["objective"].append(objective(d, x_n, b, td))
    x_next = x_n + d
    v_next = d / h
    return (x_next, v_next, history) if record else (x_next, v_next)


def eq2_residual(v_damped: np.ndarray, x_next: np.ndarray, v_next: np.ndarray,
                 f_ext: np.ndarray, td: TypeData) -> np.ndarray:
    """Residual of Eq. (2): M (v_{n+1} - v_n)/h - (F_int(x_{n+1}) + F_ext - C v_{n+1}),

    with C = (M~ - M)/h and v_n the velocity after the PBD damping operator.
    """
    C_v = (apply_M_tilde(v_next, td) - td.mass[:, None] * v_next) / td.h
    lhs = td.mass[:, None] * (v_next - v_damped) / td.h
    return lhs - (-grad_energy(x_next, td) + f_ext - C_v)


def run(x0: np.ndarray, v0: np.ndarray, forces_of_step, td: TypeData,
        n_steps: int, n_iterations: int, v_max: float = 0.0, median_filter: bool = False, collisions=None):
    """n_steps time steps; `forces_of_step(s)` returns F_ext for step s (median-filtered over the
    one-ring first if asked); v_max > 0 caps the vertex velocities."""
    x, v = x0.copy(), v0.copy()
    for s in range(n_steps):
        f = forces_of_step(s)
        if median_filter:
            f = median_filter_forces(f, td)
        x, v = step(x, v, f, td, n_iterations, v_max=v_max, collisions=collisions)
    return x, v
