"""Pins for the closing step (dual energy L100, floors L504, remedy (ii) L105) and the CFL reduction
(Eqs. 1-2) of the oracle.  CPU only."""
import math

import numpy as np
import pytest
import torch

from paper_1712_07070_b200 import inputs

G = 5.0 / 3.0
MHM, CTU, PLM, PPM, ROE, HLLC, HLLE = 1, 2, 1, 2, 1, 2, 3


def cons(rho, u, v, w, p, g=G, s=None):
    U = [rho, rho * u, rho * v, rho * w, p / (g - 1) + 0.5 * rho * (u * u + v * v + w * w)]
    if s is not None:
        U.append(s)
    return np.array(U)


def test_dual_energy_switch_closed_form(oracle_mod):
    """E_the/E_kin < xi  <=>  Mach > sqrt(2/(gamma (gamma-1) xi)) = 13.4 for gamma=5/3, xi=0.01."""
    o = oracle_mod.make_opts(n_scalar=1, dual_energy=True, de_xi=1e-2)
    rho, p = 2.0, 0.3
    cs = math.sqrt(G * p / rho)
    mach_switch = math.sqrt(2.0 / (G * (G - 1) * 1e-2))
    assert mach_switch == pytest.approx(13.416, abs=1e-3)
    s_true = p / rho ** (G - 1)
    # above the switch: E is rebuilt from the entropy, whatever E held before
    U = cons(rho, 14.0 * cs, 0, 0, p, s=s_true)
    U[4] *= 1.0 + 3e-4                                  # corrupt E (truncation error of E - E_kin)
    V, ok, st = oracle_mod.close_cell(U, G, o)
    assert ok and st["n_dual_fix"] == 1 and V[5] == U[5]
    ekin = 0.5 * U[1] ** 2 / rho
    assert V[4] == pytest.approx(ekin + p / (G - 1), rel=1e-15)
    # below the switch: E kept, entropy resynchronised from E
    U = cons(rho, 13.0 * cs, 0, 0, p, s=123.0)
    V, ok, st = oracle_mod.close_cell(U, G, o)
    assert ok and st["n_dual_fix"] == 0 and V[4] == U[4]
    assert V[5] == pytest.approx(s_true, rel=1e-11)
    # dual energy off: nothing touched
    V, ok, _ = oracle_mod.close_cell(U, G, oracle_mod.make_opts(n_scalar=1))
    assert np.array_equal(V, U)


def test_floors_closed_form(oracle_mod):
    o = oracle_mod.make_opts(min_dens=1e-3, min_pres=1e-4, min_temp=0.5)
    U = cons(1e-5, 1.0, 0, 0, 1e-9)
    V, ok, st = oracle_mod.close_cell(U, G, o)
    assert ok and st["n_floor"] == 1
    assert V[0] == 1e-3 and np.array_equal(V[1:4], U[1:4])
    ekin = 0.5 * U[1] ** 2 / 1e-3
    assert V[4] == pytest.approx(ekin + max(1e-4, 0.5 * 1e-3) / (G - 1), rel=1e-15)
    U = cons(1.0, 0.2, 0, 0, 2.0)                       # well above every floor
    V, ok, st = oracle_mod.close_cell(U, G, o)
    assert ok and st["n_floor"] == 0 and np.array_equal(V, U)
    # no floors: a negative pressure is reported, not repaired
    U = cons(1.0, 0.2, 0, 0, -0.1)
    V, ok, _ = oracle_mod.close_cell(U, G, oracle_mod.make_opts())
    assert not ok and np.array_equal(V, U)
    U[0] = float("nan")
    assert not oracle_mod.close_cell(U, G, oracle_mod.make_opts())[1]


def test_cfl_closed_forms_and_brute_force(oracle_mod):
    rho, p = 1.7, 0.6
    cs = math.sqrt(G * p / rho)
    u = np.empty((2, 5, 16, 16, 16))
    u[:] = cons(rho, 0.3, -0.9, 0.5, p)[None, :, None, None, None]
    dt, sp = oracle_mod.cfl_dt(u, 0.1, G, 0.5, MHM)
    assert sp[0] == pytest.approx(0.3 + 0.9 + 0.5 + 3 * cs, rel=1e-15)      # Eq. (2)
    assert dt == pytest.approx(0.5 * 0.1 / (1.7 + 3 * cs), rel=1e-15)
    dt, sp = oracle_mod.cfl_dt(u, 0.1, G, 0.5, CTU)
    assert sp[1] == pytest.approx(0.9 + cs, rel=1e-15)                        # Eq. (1)
    # brute force on a random field
    f = inputs.turbulence_field(16, 4, kmax=3, gamma=G)
    ui = inputs.pack_periodic(f)[:, :, 3:19, 3:19, 3:19].contiguous().numpy()
    r, vx, vy, vz = ui[:, 0], ui[:, 1] / ui[:, 0], ui[:, 2] / ui[:, 0], ui[:, 3] / ui[:, 0]
    pr = (G - 1) * (ui[:, 4] - 0.5 * r * (vx ** 2 + vy ** 2 + vz ** 2))
    c = np.sqrt(G * pr / r)
    s2 = (np.abs(vx) + np.abs(vy) + np.abs(vz) + 3 * c).max()
    s1 = (np.maximum(np.maximum(np.abs(vx), np.abs(vy)), np.abs(vz)) + c).max()
    assert oracle_mod.cfl_dt(ui, 1 / 16, G, 0.5, MHM)[0] == pytest.approx(0.5 / 16 / s2, rel=1e-13)
    assert oracle_mod.cfl_dt(ui, 1 / 16, G, 0.5, CTU)[0] == pytest.approx(0.5 / 16 / s1, rel=1e-13)


def test_fused_group_speed_equals_cfl_of_the_output(oracle_mod):
    f = inputs.turbulence_field(16, 8, kmax=3, gamma=G)
    p = inputs.pack_periodic(f).numpy()
    for scheme in (MHM, CTU):
        r = oracle_mod.fluid_advance(p, 0.003, 1 / 16, G, scheme, PLM, HLLC)
        _, sp = oracle_mod.cfl_dt(r["out"], 1 / 16, G, 0.5, scheme)
        assert np.array_equal(sp, r["speed"])


def _blast(n=16):
    one = torch.ones((n, n, n), dtype=torch.float64)
    pres = 1e-6 * one.clone()
    pres[7:9, 7:9, 7:9] = 1e3
    return inputs.prim_to_cons(one, 0 * one, 0 * one, 0 * one, pres, G)


def test_remedy_ii_first_order_recompute(oracle_mod):
    """Mach-10, sigma=2 turbulence drives some cells negative at second order; remedy (ii) (L105) must
    replace exactly those cells by the first-order unsplit Godunov update, which is checked here
    against its definition built from the (separately pinned) single-face solver."""
    f = inputs.turbulence_field(16, 3, kmax=6, gamma=G, mach=10.0, sigma=2.0)
    p = inputs.pack_periodic(f).numpy()
    dh = 1 / 16
    dt = oracle_mod.cfl_dt(inputs.interior(inputs.pack_periodic(f)).contiguous().numpy(), dh, G, 0.45, CTU)[0]
    off = oracle_mod.fluid_advance(p, dt, dh, G, CTU, PPM, HLLC, oracle_mod.make_opts())
    on = oracle_mod.fluid_advance(p, dt, dh, G, CTU, PPM, HLLC, oracle_mod.make_opts(remedy_first_order=True))
    assert off["stats"]["n_unphysical"] > 50 and off["stats"]["n_first_order"] == 0
    assert on["stats"]["n_first_order"] == off["stats"]["n_unphysical"]
    assert on["stats"]["n_unphysical"] == 0
    uo = off["out"][0]
    ekin = 0.5 * (uo[1] ** 2 + uo[2] ** 2 + uo[3] ** 2) / uo[0]
    bad = ~((uo[0] > 0) & ((uo[4] - ekin) > 0))
    assert bad.sum() == off["stats"]["n_unphysical"]
    assert np.array_equal(on["out"][0][:, ~bad], uo[:, ~bad])          # only failed cells replaced
    assert np.array_equal(on["flux"], off["flux"])                      # flux_out keeps the high-order flux
    pin = p[0]
    for k, j, i in np.argwhere(bad)[::20]:
        c = (k + 3, j + 3, i + 3)
        U0 = pin[:, c[0], c[1], c[2]]
        acc = np.zeros(5)
        for d, ax in ((0, 2), (1, 1), (2, 0)):
            lo, hi = list(c), list(c)
            lo[ax] -= 1
            hi[ax] += 1
            Fm, _ = oracle_mod.riemann(HLLC, d, pin[:, lo[0], lo[1], lo[2]], U0, G)
            Fp, _ = oracle_mod.riemann(HLLC, d, U0, pin[:, hi[0], hi[1], hi[2]], G)
            acc += Fp - Fm
        ref = U0 - dt / dh * acc
        assert np.allclose(on["out"][0][:, k, j, i], ref, rtol=1e-12, atol=1e-12 * np.abs(U0).max())


def test_pressure_floor_keeps_blast_positive(oracle_mod):
    f = _blast()
    p = inputs.pack_periodic(f).numpy()
    dh = 1 / 16
    dt = 0.45 * dh / math.sqrt(G * 1e3)
    r = oracle_mod.fluid_advance(p, dt, dh, G, MHM, PLM, HLLE, oracle_mod.make_opts(min_pres=1e-10))
    u = r["out"][0]
    pr = (G - 1) * (u[4] - 0.5 * (u[1] ** 2 + u[2] ** 2 + u[3] ** 2) / u[0])
    assert r["stats"]["n_unphysical"] == 0 and pr.min() >= 1e-10 * (1 - 1e-9) and u[0].min() > 0


def test_dual_energy_step_on_cold_supersonic_flow(oracle_mod):
    """Uniform Mach-50 flow with a density ripple: E - E_kin loses ~4 digits; with dual energy the pressure
    recovered from the output stays uniform to round-off of s, without it it does not (fp64: compare errors)."""
    n = 16
    x = (torch.arange(n, dtype=torch.float64) + 0.5) / n
    rho = (1 + 0.2 * torch.sin(2 * math.pi * x))[None, None, :].expand(n, n, n).contiguous()
    one = torch.ones_like(rho)
    cs = math.sqrt(G)
    f = inputs.prim_to_cons(rho, 50 * cs * one, 0 * one, 0 * one, one, G, entropy=True)
    p = inputs.pack_periodic(f).numpy()
    dh = 1 / n
    dt = 0.4 * dh / (51 * cs)
    o = oracle_mod.make_opts(n_scalar=1, dual_energy=True)
    r = oracle_mod.fluid_advance(p, dt, dh, G, CTU, PLM, HLLC, o)
    assert r["stats"]["n_dual_fix"] == 16 ** 3 and r["stats"]["n_unphysical"] == 0
    u = r["out"][0]
    pres_s = u[5] * u[0] ** (G - 1)
    pres_e = (G - 1) * (u[4] - 0.5 * u[1] ** 2 / u[0])
    assert np.abs(pres_e - pres_s).max() <= 1e-11          # E rebuilt from s
    # entropy advected as a passive scalar of a pure contact: P from s stays 1 up to the scheme's
    # truncation error in rho^(gamma-1) q, far below the 1e-2 the ripple itself would give
    assert np.abs(pres_s - 1.0).max() < 5e-3


def _retry_case(oracle_mod):
    """Mach-3 turbulence advanced with 5x the CFL-0.5 step of Eq. (2): the first attempts leave negative pressures."""
    f = inputs.turbulence_field(16, 3, kmax=6, gamma=G, mach=3.0, sigma=1.0)
    p = inputs.pack_periodic(f).numpy()
    dh = 1 / 16
    dt0 = 5.0 * oracle_mod.cfl_dt(inputs.interior(inputs.pack_periodic(f)).contiguous().numpy(), dh, G, 0.5, MHM)[0]
    return p, dt0, dh


def test_remedy_iv_v_retry_loop(oracle_mod):
    """Remedies (iv), (v) (L107-108), pinned by what the text fixes: the accepted step is dt0 * 0.8^k with k the SMALLEST
    count whose attempt has no unphysical cell (every earlier attempt, recomputed here by direct calls, has some); the
    result is the direct call at that step, from the same input; a physical first attempt is returned untouched with
    k = 0; and the loop aborts once the reduced step falls below dt_min."""
    p, dt0, dh = _retry_case(oracle_mod)
    r = oracle_mod.fluid_advance_retry(p, dt0, dh, G, MHM, PLM, ROE)
    k = r["n_retries"]
    assert k >= 2 and r["stats"]["n_unphysical"] == 0
    dt = dt0
    for _ in range(k):
        assert oracle_mod.fluid_advance(p, dt, dh, G, MHM, PLM, ROE)["stats"]["n_unphysical"] > 0
        dt = dt * 0.8
    assert r["dt_used"] == dt and abs(dt / dt0 - 0.8 ** k) < 1e-14
    direct = oracle_mod.fluid_advance(p, dt, dh, G, MHM, PLM, ROE)
    assert np.array_equal(direct["out"], r["out"]) and np.array_equal(direct["flux"], r["flux"])
    uo = r["out"][0]
    assert uo[0].min() > 0 and (uo[4] - 0.5 * (uo[1] ** 2 + uo[2] ** 2 + uo[3] ** 2) / uo[0]).min() > 0
    # another ratio: fewer, larger reductions
    r2 = oracle_mod.fluid_advance_retry(p, dt0, dh, G, MHM, PLM, ROE, dt_ratio=0.5)
    assert 1 <= r2["n_retries"] < k and r2["dt_used"] == dt0 * 0.5 ** r2["n_retries"]
    # physical first attempt
    r0 = oracle_mod.fluid_advance_retry(p, dt0 / 5.0, dh, G, MHM, PLM, ROE)
    assert r0["n_retries"] == 0 and r0["dt_used"] == dt0 / 5.0
    assert np.array_equal(r0["out"], oracle_mod.fluid_advance(p, dt0 / 5.0, dh, G, MHM, PLM, ROE)["out"])
    # (v): abort at the threshold -- the last allowed attempt is the largest dt0 * 0.8^j >= dt_min
    with pytest.raises(FloatingPointError):
        oracle_mod.fluid_advance_retry(p, dt0, dh, G, MHM, PLM, ROE, dt_min=dt * 1.01)
    assert oracle_mod.fluid_advance_retry(p, dt0, dh, G, MHM, PLM, ROE, dt_min=dt * 0.99)["n_retries"] == k
