"""Pins for oracle.fill_ghosts (the same-level ghost filling with the boundary conditions of PAPER.md L98 that the
CUDA refresh kernel is compared with): periodic = the independent torch gather of inputs.pack_periodic; outflow =
zero gradient across the face; reflecting = a state that is mirror-symmetric about the face (normal momentum odd) is
its own ghost image, and the normal momentum of mirrored cells is negated; interior cells are never changed."""
import numpy as np
import torch

from paper_1712_07070_b200 import inputs


def _field(seed=3, shape=(32, 48, 16)):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((5,) + shape) + np.array([3.0, 0, 0, 0, 5.0])[:, None, None, None]


def test_periodic_is_pack_periodic(oracle_mod):
    f = _field()
    got = oracle_mod.fill_ghosts(f)
    ref = inputs.pack_periodic(torch.from_numpy(f)).numpy()
    assert np.array_equal(got, ref)


def test_outflow_and_reflecting(oracle_mod):
    f = _field()
    O, R, P = oracle_mod.OUTFLOW, oracle_mod.REFLECTING, oracle_mod.PERIODIC
    got = oracle_mod.fill_ghosts(f, bc=((O, R), (R, O), (P, P)))
    gz, gy, gx = 2, 3, 1
    g = got.reshape(gz, gy, gx, 5, 22, 22, 22)
    # interior untouched
    assert np.array_equal(inputs.unpack(torch.from_numpy(np.ascontiguousarray(got[..., 3:19, 3:19, 3:19])), gz, gy, gx).numpy(), f)
    # x low: outflow -> the three ghost layers repeat the first interior layer (same y, z line of the padded group)
    for l in range(3):
        assert np.array_equal(g[:, :, 0, :, :, :, l], g[:, :, 0, :, :, :, 3])
    # x high: reflecting -> ghost layer 19+l mirrors interior layer 18-l, x momentum negated, the rest equal
    for l in range(3):
        a, b = g[:, :, 0, :, :, :, 19 + l], g[:, :, 0, :, :, :, 18 - l]
        assert np.array_equal(a[:, :, 1], -b[:, :, 1])
        assert np.array_equal(a[:, :, [0, 2, 3, 4]], b[:, :, [0, 2, 3, 4]])
    # y low: reflecting (y momentum odd), y high: outflow
    for l in range(3):
        a, b = g[:, 0, :, :, :, 2 - l, :], g[:, 0, :, :, :, 3 + l, :]
        assert np.array_equal(a[:, :, 2], -b[:, :, 2]) and np.array_equal(a[:, :, [0, 1, 3, 4]], b[:, :, [0, 1, 3, 4]])
        assert np.array_equal(g[:, gy - 1, :, :, :, 19 + l, :], g[:, gy - 1, :, :, :, 18, :])
    # z: periodic wrap
    assert np.array_equal(g[0, :, :, :, 0:3], g[gz - 1, :, :, :, 16:19])
    # a field that is mirror symmetric about the reflecting x-high wall is continued smoothly: ghosts == the mirrored
    # interior means a symmetric scalar has zero normal gradient at the wall
    assert np.array_equal(g[:, :, 0, 0, :, :, 19], g[:, :, 0, 0, :, :, 18])


def test_reflecting_box_is_closed_and_outflow_lets_a_pulse_leave(oracle_mod):
    """Physics pin of the boundary conditions through the oracle solver: in a box with reflecting walls on all six
    sides no mass or energy crosses the walls (the Riemann problem between a state and its mirror image has zero mass
    and energy flux), so both totals stay constant to round-off over several steps of a sloshing gas, while with
    outflow walls the same gas loses mass."""
    n, gamma = 32, 1.4
    dh = 1.0 / n
    z, y, x = np.meshgrid(*(3 * [(np.arange(n) + 0.5) * dh]), indexing="ij")
    rho = 1.0 + 0.5 * np.exp(-((x - 0.3) ** 2 + (y - 0.6) ** 2 + (z - 0.5) ** 2) / 0.02)
    vx, vy, vz = 0.8 * np.ones_like(rho), -0.5 * np.ones_like(rho), 0.3 * np.ones_like(rho)
    pres = np.ones_like(rho)
    u = np.stack([rho, rho * vx, rho * vy, rho * vz, pres / (gamma - 1) + 0.5 * rho * (vx ** 2 + vy ** 2 + vz ** 2)])
    R, O = oracle_mod.REFLECTING, oracle_mod.OUTFLOW

    def run(bc, steps=4):
        f = u.copy()
        for _ in range(steps):
            padded = oracle_mod.fill_ghosts(f, bc)
            dt = oracle_mod.cfl_dt(np.ascontiguousarray(padded[..., 3:19, 3:19, 3:19]), dh, gamma, 0.4, 1)[0]
            out = oracle_mod.fluid_advance(padded, dt, dh, gamma, 1, 1, 3, want_flux=False)["out"]
            f = inputs.unpack(torch.from_numpy(out), 2, 2, 2).numpy()
        return f

    closed = run(((R, R),) * 3)
    assert abs(closed[0].sum() - u[0].sum()) <= 1e-13 * u[0].sum()
    assert abs(closed[4].sum() - u[4].sum()) <= 1e-13 * u[4].sum()
    assert np.abs(closed[0] - u[0]).max() > 1e-3                  # the gas did move
    opened = run(((O, O),) * 3)
    assert abs(opened[0].sum() - u[0].sum()) > 1e-7 * u[0].sum()       # in- and outflow nearly cancel, but not to round-off
    assert np.abs(opened[0] - closed[0]).max() > 1e-3                  # and the walls do matter


def test_table_driven_sibling_copy(oracle_mod):
    """oracle.fill_ghosts_table: with the periodic table of a 2 x 3 x 1 box it is pack_periodic; with some entries
    set to -1 exactly those slabs keep their previous content."""
    f = _field()
    gz, gy, gx = 2, 3, 1
    u = inputs.interior(inputs.pack_periodic(torch.from_numpy(f))).contiguous().numpy()
    nbr = np.empty((6, 27), dtype=np.int32)
    for g in range(6):
        bz, by, bx = g // (gy * gx), (g // gx) % gy, g % gx
        for k in range(27):
            dz, dy, dx = k // 9 - 1, (k // 3) % 3 - 1, k % 3 - 1
            nbr[g, k] = (((bz + dz) % gz) * gy + (by + dy) % gy) * gx + (bx + dx) % gx
    full = oracle_mod.fill_ghosts_table(u, nbr, np.full((6, 5, 22, 22, 22), np.nan))
    assert np.array_equal(full, inputs.pack_periodic(torch.from_numpy(f)).numpy())
    nbr2 = nbr.copy()
    nbr2[:, 14] = -1                       # no +x neighbour anywhere
    nbr2[3, 4] = -1                        # group 3: no (dz, dy, dx) = (-1, 0, 0) neighbour
    part = oracle_mod.fill_ghosts_table(u, nbr2, np.full((6, 5, 22, 22, 22), np.nan))
    hole = np.isnan(part)
    assert hole[:, :, 3:19, 3:19, 19:22].all() and hole[3, :, 0:3, 3:19, 3:19].all()
    assert hole.sum() == 6 * 5 * 16 * 16 * 3 + 5 * 3 * 16 * 16
    assert np.array_equal(part[~hole], full[~hole])
