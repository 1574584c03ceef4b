"""Pins for the oracle's Riemann solvers (oracle/hydro_oracle.c O5) -- CPU only."""
import math

import numpy as np
import pytest

import exact_riemann as er
from helpers import load_golden

G = 1.4


def cons(rho, u, v, w, p, g=G):
    return np.array([rho, rho * u, rho * v, rho * w, p / (g - 1) + 0.5 * rho * (u * u + v * v + w * w)])


def xflux(rho, u, v, w, p, g=G):
    e = p / (g - 1) + 0.5 * rho * (u * u + v * v + w * w)
    return np.array([rho * u, rho * u * u + p, rho * u * v, rho * u * w, u * (e + p)])


def test_exact_solver_matches_printed_sod_values():
    gold = load_golden("sod_exact.txt")
    ps, us = er.star_state(1, 0, 1, 0.125, 0, 0.1, G)
    assert abs(ps - gold["p_star"]) < 2e-10 and abs(us - gold["u_star"]) < 2e-10
    rho, _, _ = er.sample(1, 0, 1, 0.125, 0, 0.1, G, np.array([0.5, 1.0]))
    assert abs(rho[0] - gold["rho_star_L"]) < 2e-10 and abs(rho[1] - gold["rho_star_R"]) < 2e-10
    rho, _, _ = er.sample(1, 0, 1, 0.125, 0, 0.1, G, np.array([gold["shock_speed"] - 1e-6, gold["shock_speed"] + 1e-6]))
    assert abs(rho[0] - gold["rho_star_R"]) < 1e-9 and rho[1] == 0.125
    f = er.godunov_flux(1, 0, 0, 0, 1, 0.125, 0, 0, 0, 0.1, G)
    assert np.allclose(f, [gold["flux_mass"], gold["flux_momx"], 0, 0, gold["flux_ener"]], atol=2e-10)


@pytest.mark.parametrize("solver", [1, 2, 3, 4])
def test_consistency_is_bitwise_for_identical_states(oracle_mod, solver):
    rng = np.random.default_rng(3)
    for _ in range(20):
        rho, p = rng.uniform(0.1, 3), rng.uniform(0.1, 3)
        u, v, w = rng.normal(size=3) * 2
        U = cons(rho, u, v, w, p)
        F, fb = oracle_mod.riemann(solver, 0, U, U, G)
        assert fb == 0
        ref = xflux(rho, u, v, w, p)
        if solver == 1:
            # dU = 0: every wave strength vanishes; F = (F+F)/2 exactly as the oracle forms F(U)
            assert np.allclose(F, ref, rtol=1e-15, atol=1e-15)
        assert np.allclose(F, ref, rtol=1e-13, atol=1e-13)


def test_roe_identities(oracle_mod):
    """sum a_k K_k = dU and sum lambda_k a_k K_k = F_R - F_L (Roe 1981, property U)."""
    rng = np.random.default_rng(11)
    for _ in range(50):
        l = (rng.uniform(0.1, 3), *(rng.normal(size=3)), rng.uniform(0.1, 3))
        r = (rng.uniform(0.1, 3), *(rng.normal(size=3)), rng.uniform(0.1, 3))
        UL, UR = cons(*l), cons(*r)
        alpha, lam, K = oracle_mod.roe_decomposition(UL, UR, G)
        scale = np.abs(UL) + np.abs(UR) + 1.0
        assert np.all(np.abs(alpha @ K - (UR - UL)) <= 2e-14 * scale)
        dF = xflux(*r) - xflux(*l)
        fscale = np.abs(xflux(*r)) + np.abs(xflux(*l)) + 1.0
        assert np.all(np.abs((alpha * lam) @ K - dF) <= 1e-13 * fscale)
        # and the Roe flux is the one-sided form F_L + sum_{lambda<0} lambda a K
        F, fb = oracle_mod.riemann(1, 0, UL, UR, G)
        if fb == 0:
            one_sided = xflux(*l) + ((alpha * np.minimum(lam, 0.0)) @ K)
            assert np.all(np.abs(F - one_sided) <= 1e-13 * fscale)


@pytest.mark.parametrize("solver", [1, 2, 3, 4])
def test_supersonic_upwinding(oracle_mod, solver):
    l, r = (1.0, 5.0, 0.3, -0.2, 1.0), (0.7, 4.5, -0.1, 0.4, 0.8)
    F, _ = oracle_mod.riemann(solver, 0, cons(*l), cons(*r), G)
    assert np.allclose(F, xflux(*l), rtol=1e-13)
    l2, r2 = (1.0, -5.0, 0.3, -0.2, 1.0), (0.7, -4.5, -0.1, 0.4, 0.8)
    F, _ = oracle_mod.riemann(solver, 0, cons(*l2), cons(*r2), G)
    assert np.allclose(F, xflux(*r2), rtol=1e-13)


def test_stationary_contact(oracle_mod):
    UL, UR = cons(1.0, 0, 0, 0, 0.7), cons(0.25, 0, 0, 0, 0.7)
    for solver in (1, 2):       # Roe and HLLC keep an isolated stationary contact exactly
        F, _ = oracle_mod.riemann(solver, 0, UL, UR, G)
        assert np.allclose(F, [0, 0.7, 0, 0, 0], atol=1e-15)
    # HLLE smears it: closed-form diffusive flux b+ b- (U_R - U_L)/(b+ - b-), b from the faster side
    F, _ = oracle_mod.riemann(3, 0, UL, UR, G)
    cl, cr = math.sqrt(G * 0.7 / 1.0), math.sqrt(G * 0.7 / 0.25)
    wl, wr = 1.0, 0.5
    Hl = (UL[4] + 0.7) / 1.0
    Hr = (UR[4] + 0.7) / 0.25
    a_roe = math.sqrt((G - 1) * (wl * Hl + wr * Hr) / (wl + wr))
    bm, bp = min(-a_roe, -cl), max(a_roe, cr)
    assert F[0] == pytest.approx(bp * bm * (0.25 - 1.0) / (bp - bm), rel=1e-13)
    assert F[0] > 0 and F[1] == pytest.approx(0.7, rel=1e-13)


@pytest.mark.parametrize("solver", [1, 2, 3])
def test_weak_jump_matches_exact_godunov_flux_to_second_order(oracle_mod, solver):
    """For a jump of size eps every approximate solver agrees with the exact Godunov flux up to
    O(eps^2): catches wrong signs / indices in any flux component, transverse ones included."""
    base = np.array([1.0, 0.3, -0.4, 0.25, 0.9])
    dirn = np.array([0.4, -0.5, 0.7, -0.3, 0.6])
    errs = []
    for eps in (1e-2, 1e-3):
        l, r = base - 0.5 * eps * dirn, base + 0.5 * eps * dirn
        F, _ = oracle_mod.riemann(solver, 0, cons(*l), cons(*r), G)
        Fe = er.godunov_flux(l[0], l[1], l[2], l[3], l[4], r[0], r[1], r[2], r[3], r[4], G)
        errs.append(np.abs(F - Fe).max())
    if solver == 3:
        # HLLE has no contact wave: the transverse/entropy jump is smeared at first order in eps
        assert errs[0] < 0.6e-2 and errs[1] < 0.6e-3
    else:
        assert errs[0] < 3e-4 and errs[1] < 3e-6, errs
        assert errs[1] < errs[0] / 50


@pytest.mark.parametrize("solver", [1, 2, 3])
def test_sod_flux_near_exact(oracle_mod, solver):
    gold = load_golden("sod_exact.txt")
    F, fb = oracle_mod.riemann(solver, 0, cons(1, 0, 0, 0, 1), cons(0.125, 0, 0, 0, 0.1), G)
    assert fb == 0
    assert abs(F[0] - gold["flux_mass"]) < 0.3 * gold["flux_mass"]
    assert abs(F[1] - gold["flux_momx"]) < 0.3 * gold["flux_momx"]
    assert abs(F[4] - gold["flux_ener"]) < 0.3 * gold["flux_ener"]
    assert F[2] == 0 and F[3] == 0


@pytest.mark.parametrize("solver", [1, 2, 3, 4])
def test_axis_rotation(oracle_mod, solver):
    """Flux through a y- (z-) face = x-face flux of the cyclically permuted states, permuted back."""
    l, r = (1.0, 0.3, -0.4, 0.25, 0.9), (0.6, -0.2, 0.5, 0.1, 0.5)
    Fx, _ = oracle_mod.riemann(solver, 0, cons(*l), cons(*r), G)
    # y-normal: normal velocity = vy, transverse (vz, vx)
    ly = (l[0], l[3], l[1], l[2], l[4])   # (rho, vx, vy, vz) with vy=l.u, vz=l.v, vx=l.w
    ry = (r[0], r[3], r[1], r[2], r[4])
    Fy, _ = oracle_mod.riemann(solver, 1, cons(*ly), cons(*ry), G)
    assert np.array_equal(Fy[[0, 2, 3, 1, 4]], Fx)
    lz = (l[0], l[2], l[3], l[1], l[4])
    rz = (r[0], r[2], r[3], r[1], r[4])
    Fz, _ = oracle_mod.riemann(solver, 2, cons(*lz), cons(*rz), G)
    assert np.array_equal(Fz[[0, 3, 1, 2, 4]], Fx)


@pytest.mark.parametrize("solver", [1, 2, 3, 4])
def test_mirror_symmetry(oracle_mod, solver):
    l, r = (1.0, 0.3, -0.4, 0.25, 0.9), (0.6, -0.2, 0.5, 0.1, 0.5)
    F, _ = oracle_mod.riemann(solver, 0, cons(*l), cons(*r), G)
    lm, rm = (r[0], -r[1], r[2], r[3], r[4]), (l[0], -l[1], l[2], l[3], l[4])
    Fm, _ = oracle_mod.riemann(solver, 0, cons(*lm), cons(*rm), G)
    assert np.allclose(Fm * np.array([-1, 1, -1, -1, -1]), F, rtol=1e-13, atol=1e-15)


@pytest.mark.parametrize("solver", [1, 2, 3, 4])
def test_scalar_flux_is_upwinded_on_mass_flux(oracle_mod, solver):
    UL = np.append(cons(1.0, 0.3, 0, 0, 0.9), 1.0 * 2.0)     # q_L = 2
    UR = np.append(cons(0.6, 0.2, 0, 0, 0.5), 0.6 * 5.0)     # q_R = 5
    F, _ = oracle_mod.riemann(solver, 0, UL, UR, G, n_scalar=1)
    assert F[0] > 0 and F[5] == F[0] * 2.0
    UL[1], UR[1] = -1.0 * 0.9, -0.6 * 0.9
    UL[4], UR[4] = cons(1.0, -0.9, 0, 0, 0.9)[4], cons(0.6, -0.9, 0, 0, 0.5)[4]
    F, _ = oracle_mod.riemann(solver, 0, UL, UR, G, n_scalar=1)
    assert F[0] < 0 and F[5] == F[0] * 5.0


def test_remedy_i_roe_falls_back_to_hlle_on_strong_rarefaction(oracle_mod):
    """Einfeldt's 1-2-3 problem: the linearised Roe intermediate states are unphysical (L104)."""
    UL, UR = cons(1.0, -2.0, 0, 0, 0.4), cons(1.0, 2.0, 0, 0, 0.4)
    F, fb = oracle_mod.riemann(1, 0, UL, UR, G)
    Fe, _ = oracle_mod.riemann(3, 0, UL, UR, G)
    assert fb == 1 and np.array_equal(F, Fe)
    # by symmetry of the 1-2-3 problem the exact mass and energy fluxes vanish
    assert abs(F[0]) < 1e-14 and abs(F[4]) < 1e-14
    # a mild problem must not take the fallback
    _, fb = oracle_mod.riemann(1, 0, cons(1, 0, 0, 0, 1), cons(0.125, 0, 0, 0, 0.1), G)
    assert fb == 0


def test_exact_solver_of_the_oracle_matches_the_test_side_solver(oracle_mod):
    """Solver 4 (Toro ch. 4) against tests/exact_riemann.py -- an independent implementation with another
    first guess and a 1e-15 stopping rule, itself pinned to the printed Sod values: the printed Godunov flux of the Sod
    problem to 1e-9, and the flux of random subsonic / supersonic / strong-shock / strong-rarefaction data, transverse
    components included, to 1e-9 of its scale (the oracle stops one Newton step after a 1e-6 change)."""
    gold = load_golden("sod_exact.txt")
    F, fb = oracle_mod.riemann(4, 0, cons(1, 0, 0, 0, 1), cons(0.125, 0, 0, 0, 0.1), G)
    assert fb == 0
    assert np.allclose(F, [gold["flux_mass"], gold["flux_momx"], 0, 0, gold["flux_ener"]], atol=1e-9)
    rng = np.random.default_rng(11)
    for k in range(300):
        rl, rr = rng.uniform(0.05, 5, size=2)
        pl, pr = 10 ** rng.uniform(-2, 2, size=2)
        ul, ur = rng.normal(size=2) * rng.choice([0.3, 3.0])
        vl, wl, vr, wr = rng.normal(size=4)
        if 2 * (math.sqrt(G * pl / rl) + math.sqrt(G * pr / rr)) / (G - 1) <= ur - ul:
            continue                                      # vacuum: covered below
        F, fb = oracle_mod.riemann(4, 0, cons(rl, ul, vl, wl, pl), cons(rr, ur, vr, wr, pr), G)
        Fe = er.godunov_flux(rl, ul, vl, wl, pl, rr, ur, vr, wr, pr, G)
        assert fb == 0
        assert np.abs(F - Fe).max() <= 1e-9 * (np.abs(Fe).max() + 1.0), (k, F, Fe)
    # data that generate vacuum (Toro eq. 4.40) are reported and handed to HLLE
    F, fb = oracle_mod.riemann(4, 0, cons(1, -20, 0, 0, 0.4), cons(1, 20, 0, 0, 0.4), G)
    Fh, _ = oracle_mod.riemann(3, 0, cons(1, -20, 0, 0, 0.4), cons(1, 20, 0, 0, 0.4), G)
    assert fb == 1 and np.array_equal(F, Fh)
