"""Pins for the oracle's SOR Poisson solver.  CPU only."""
import numpy as np
import pytest
import scipy.sparse as sp
import scipy.sparse.linalg as spla


def _problem(seed, n=3):
    rng = np.random.default_rng(seed)
    phi = rng.standard_normal((n, 18, 18, 18))
    rho = rng.standard_normal((n, 16, 16, 16)) + 2.0
    return phi, rho


def _direct(phi, rho, dh, coeff):
    """The discrete Dirichlet problem solved without any relaxation: 7-point matrix on the 16^3 unknowns, boundary
    values moved to the right-hand side, sparse LU."""
    n = 16
    e = sp.eye(n)
    d = sp.diags([1.0, -2.0, 1.0], [-1, 0, 1], shape=(n, n))
    A = (sp.kron(sp.kron(d, e), e) + sp.kron(sp.kron(e, d), e) + sp.kron(sp.kron(e, e), d)).tocsc()
    lu = spla.splu(A)
    out = phi.copy()
    for p in range(phi.shape[0]):
        b = coeff * dh * dh * rho[p].copy()
        b[0] -= phi[p, 0, 1:17, 1:17]
        b[-1] -= phi[p, 17, 1:17, 1:17]
        b[:, 0] -= phi[p, 1:17, 0, 1:17]
        b[:, -1] -= phi[p, 1:17, 17, 1:17]
        b[:, :, 0] -= phi[p, 1:17, 1:17, 0]
        b[:, :, -1] -= phi[p, 1:17, 1:17, 17]
        out[p, 1:17, 1:17, 1:17] = lu.solve(b.ravel()).reshape(n, n, n)
    return out


def test_sor_converges_to_the_direct_solution_of_the_discrete_problem(oracle_mod):
    """"solve the discretized Poisson equation to machine precision" (L126): enough SOR iterations reach the sparse-LU solution
    of the same 7-point Dirichlet problem; the boundary layer never changes; fewer iterations are further away."""
    phi0, rho = _problem(1)
    dh, coeff = 0.37, 4 * np.pi * 0.8
    omega = 2.0 / (1.0 + np.sin(np.pi / 17))                    # optimal SOR parameter of a 16-cell Dirichlet box (Press et al.)
    want = _direct(phi0, rho, dh, coeff)
    phi, _ = oracle_mod.poisson_sor(phi0, rho, dh, coeff, omega, 200)
    scale = np.abs(want).max()
    assert np.abs(phi - want).max() <= 1e-12 * scale
    edge = np.ones((18, 18, 18), bool)
    edge[1:17, 1:17, 1:17] = False
    assert np.array_equal(phi[:, edge], phi0[:, edge])
    e10 = np.abs(oracle_mod.poisson_sor(phi0, rho, dh, coeff, omega, 10)[0] - want).max()
    e40 = np.abs(oracle_mod.poisson_sor(phi0, rho, dh, coeff, omega, 40)[0] - want).max()
    assert e10 > e40 > 1e-9 * scale
    # omega = 1 is Gauss-Seidel: converges too, far more slowly (the reason for over-relaxation)
    gs = np.abs(oracle_mod.poisson_sor(phi0, rho, dh, coeff, 1.0, 40)[0] - want).max()
    assert gs > 100 * e40


def test_sor_fixed_point_sweep_definition_and_acceleration(oracle_mod):
    """(a) A quadratic potential is an exact solution of the 7-point equation (laplacian of x^2 + 2 y^2 - z^2 = 4): with
    rho = 4 / coeff it is a fixed point of every sweep, and its central-difference acceleration is the exact gradient.
    (b) One iteration written out cell by cell in plain loops (red cells first, each using the latest neighbours)."""
    dh, coeff, omega = 0.5, 2.5, 1.6
    x = (np.arange(18) - 8.5) * dh
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    quad = (X ** 2 + 2 * Y ** 2 - Z ** 2 + 0.3 * X - 0.7 * Z + 1.0)[None]
    rho = np.full((1, 16, 16, 16), 4.0 / coeff)
    phi, acc = oracle_mod.poisson_sor(quad, rho, dh, coeff, omega, 7)
    assert np.abs(phi - quad).max() <= 1e-12 * np.abs(quad).max()
    a = slice(5, 13)
    assert np.abs(acc[0, 0] + (2 * X + 0.3)[a, a, a]).max() <= 1e-12
    assert np.abs(acc[0, 1] + (4 * Y)[a, a, a]).max() <= 1e-12
    assert np.abs(acc[0, 2] + (-2 * Z - 0.7)[a, a, a]).max() <= 1e-12
    phi0, rho = _problem(2, n=1)
    p = phi0[0].copy()
    for colour in (0, 1):
        for k in range(1, 17):
            for j in range(1, 17):
                for i in range(1, 17):
                    if (i + j + k) % 2 == colour:
                        r = (p[k, j, i - 1] + p[k, j, i + 1] + p[k, j - 1, i] + p[k, j + 1, i] + p[k - 1, j, i] + p[k + 1, j, i]
                             - 6 * p[k, j, i] - coeff * dh * dh * rho[0, k - 1, j - 1, i - 1])
                        p[k, j, i] += omega * r / 6
    got, _ = oracle_mod.poisson_sor(phi0, rho, dh, coeff, omega, 1, want_acc=False)
    assert np.abs(got[0] - p).max() <= 1e-14 * np.abs(p).max()


def test_residual_definition_and_decay(oracle_mod):
    """poisson_residual: zero for the quadratic exact solution and (to round-off) for the sparse-LU solution; equal to the defect
    of one cell written out by hand when a single cell of an exact solution is perturbed (the cell itself sees -6 eps, its six
    neighbours +eps); monotonically smaller as SOR proceeds."""
    dh, coeff = 0.5, 2.5
    x = (np.arange(18) - 8.5) * dh
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    quad = (X ** 2 + 2 * Y ** 2 - Z ** 2)[None]
    rho = np.full((1, 16, 16, 16), 4.0 / coeff)
    assert oracle_mod.poisson_residual(quad, rho, dh, coeff)[0] <= 1e-12
    bumped = quad.copy()
    bumped[0, 7, 9, 4] += 0.125
    assert abs(oracle_mod.poisson_residual(bumped, rho, dh, coeff)[0] - 6 * 0.125) <= 1e-12
    bumped = quad.copy()
    bumped[0, 0, 9, 4] += 0.125                                   # a boundary cell: only its one inner neighbour sees it
    assert abs(oracle_mod.poisson_residual(bumped, rho, dh, coeff)[0] - 0.125) <= 1e-12
    phi0, rho = _problem(3)
    omega = 2.0 / (1.0 + np.sin(np.pi / 17))
    res = [oracle_mod.poisson_residual(oracle_mod.poisson_sor(phi0, rho, dh, coeff, omega, n, want_acc=False)[0], rho, dh, coeff).max()
           for n in (0, 5, 20, 60, 200)]
    assert all(a > b for a, b in zip(res, res[1:])) and res[-1] <= 1e-12 * np.abs(phi0).max()
    assert oracle_mod.poisson_residual(_direct(phi0, rho, dh, coeff), rho, dh, coeff).max() <= 1e-12 * np.abs(phi0).max()


# ---------------------------------------------------------------------------------------------------------------
# fluid gravity update behind the Poisson solve (R28)
# ---------------------------------------------------------------------------------------------------------------
def _gas(g=2, seed=3, nv=5):
    rng = np.random.default_rng(seed)
    u = np.empty((g, nv, 16, 16, 16))
    u[:, 0] = rng.uniform(0.5, 2.0, (g, 16, 16, 16))
    v = rng.normal(0, 0.5, (g, 3, 16, 16, 16))
    p = rng.uniform(0.5, 2.0, (g, 16, 16, 16))
    u[:, 1:4] = u[:, 0:1] * v
    u[:, 4] = p / (5 / 3 - 1) + 0.5 * u[:, 0] * (v ** 2).sum(axis=1)
    if nv > 5:
        u[:, 5:] = rng.uniform(0.1, 1.0, (g, nv - 5, 16, 16, 16))
    return u


def test_gravity_update_closed_forms(oracle_mod):
    """Uniform acceleration: momentum gains dt rho g exactly as written; the thermal energy E - |m|^2 / 2 rho is unchanged
    to round-off (the energy correction is the kinetic-energy difference); density and scalars untouched bit for bit;
    a kick followed by the opposite kick restores the state; N kicks of a gas at rest give v = N dt g."""
    u = _gas(nv=7)
    gvec = np.array([0.3, -0.7, 1.1])
    acc = np.broadcast_to(gvec[None, :, None, None, None], (16, 3, 8, 8, 8)).copy()
    dt = 0.05
    new = oracle_mod.gravity_update(u, acc, dt)
    assert np.array_equal(new[:, 0], u[:, 0]) and np.array_equal(new[:, 5:], u[:, 5:])
    for d in range(3):
        assert np.array_equal(new[:, 1 + d], u[:, 1 + d] + (dt * u[:, 0]) * gvec[d])
    eth = lambda a: a[:, 4] - 0.5 * (a[:, 1:4] ** 2).sum(axis=1) / a[:, 0]
    assert np.abs(eth(new) - eth(u)).max() <= 2e-15 * np.abs(u[:, 4]).max()
    back = oracle_mod.gravity_update(new, -acc, dt)
    assert np.abs(back - u).max() <= 4e-15 * np.abs(u).max()
    rest = _gas()
    rest[:, 1:4] = 0.0
    rest[:, 4] = 1.5
    cur = rest
    for _ in range(8):
        cur = oracle_mod.gravity_update(cur, acc, dt)
    for d in range(3):
        assert np.abs(cur[:, 1 + d] / cur[:, 0] - 8 * dt * gvec[d]).max() <= 1e-14
    assert np.abs(cur[:, 4] - (1.5 + 0.5 * cur[:, 0] * ((8 * dt * gvec) ** 2).sum())).max() <= 1e-13


def test_gravity_update_patch_to_group_mapping(oracle_mod):
    """acc lives in the patch layout of poisson_sor (patch n = 8 g + oz*4 + oy*2 + ox), the fluid in the group layout: a
    kick confined to one patch changes exactly that octant of that group, with the patch's own cell order."""
    u = _gas(g=3)
    acc = np.zeros((24, 3, 8, 8, 8))
    n = 8 * 1 + (1 * 4 + 0 * 2 + 1)                      # group 1, octant oz=1, oy=0, ox=1
    acc[n, 0] = np.arange(512).reshape(8, 8, 8)          # distinct value per cell: x fastest
    new = oracle_mod.gravity_update(u, acc, 1.0)
    diff = new != u
    assert not diff[0].any() and not diff[2].any()
    box = np.zeros((16, 16, 16), dtype=bool)
    box[8:16, 0:8, 8:16] = True                          # [z, y, x]
    assert not diff[1][:, ~box].any() and not diff[1, 0].any() and not diff[1, 2:4].any()
    dm = (new[1, 1] - u[1, 1]) / u[1, 0]
    assert dm[8, 0, 9] == pytest.approx(1.0, rel=1e-14) and dm[9, 0, 8] == pytest.approx(64.0, rel=1e-14) and dm[8, 1, 8] == pytest.approx(8.0, rel=1e-14)
