"""Pins for slope limiters, PLM/PPM face values and characteristic tracing (oracle O2, O3, O4-CTU(a))."""
import math

import numpy as np
import pytest

PLM, PPM = 1, 2


def test_generalized_minmod_closed_forms(oracle_mod):
    o = oracle_mod
    assert o.limited_slope(1, 1.0, 1.0, 3.0) == 1.0          # theta=1: plain minmod
    assert o.limited_slope(1, 1.0, -3.0, -1.0) == -1.0
    assert o.limited_slope(1, 2.0, 1.0, 3.0) == 2.0          # theta=2: min(2, 2, 6)
    assert o.limited_slope(1, 2.0, 1.0, 1.5) == 1.25         # centred slope wins
    assert o.limited_slope(1, 1.5, 1.0, 100.0) == 1.5
    for th in (1.0, 1.5, 2.0):
        assert o.limited_slope(1, th, 1.0, -1.0) == 0.0      # extremum
        assert o.limited_slope(1, th, 0.0, 1.0) == 0.0       # tie at zero -> 0
        assert o.limited_slope(1, th, 0.7, 0.7) == pytest.approx(0.7, rel=1e-15)
    assert o.limited_slope(2, 0, 1.0, 3.0) == pytest.approx(1.5)        # van Leer: harmonic mean
    assert o.limited_slope(3, 0, 1.0, 3.0) == pytest.approx(12.0 / 10.0)  # van Albada
    assert o.limited_slope(2, 0, 1.0, -3.0) == 0.0 and o.limited_slope(3, 0, -1.0, 3.0) == 0.0


@pytest.mark.parametrize("recon", [PLM, PPM])
def test_linear_data_reproduced_exactly(oracle_mod, recon):
    a, b = 0.75, -0.125       # exactly representable
    w = np.array([a + b * i for i in range(-2, 3)])
    wm, wp = oracle_mod.face_values(recon, w)
    assert wm == a - 0.5 * b and wp == a + 0.5 * b


def test_ppm_interface_value_is_exact_for_cubic_cell_averages(oracle_mod):
    """Colella & Woodward (1984) eq. 1.6 is fourth order: exact for cell averages of a cubic, when the
    limiter is inactive (gentle monotone profile)."""
    c0, c1, c2, c3 = 1.0, 0.5, 0.02, 0.003

    def avg(i):   # cell average of the cubic over [i-1/2, i+1/2]
        F = lambda x: c0 * x + c1 * x ** 2 / 2 + c2 * x ** 3 / 3 + c3 * x ** 4 / 4
        return F(i + 0.5) - F(i - 0.5)

    w = np.array([avg(i) for i in range(-2, 3)])
    wm, wp = oracle_mod.face_values(PPM, w)
    point = lambda x: c0 + c1 * x + c2 * x ** 2 + c3 * x ** 3
    # the gen.-minmod(2) slope equals the centred difference here, which is what eq. 1.6 assumes
    assert wp == pytest.approx(point(0.5), abs=2e-15 + 0.0)
    assert wm == pytest.approx(point(-0.5), abs=2e-15 + 0.0)


@pytest.mark.parametrize("recon", [PLM, PPM])
def test_face_values_monotone_and_extrema_flattened(oracle_mod, recon):
    rng = np.random.default_rng(5)
    for _ in range(300):
        w = np.sort(rng.uniform(0, 1, 5)) if rng.uniform() < 0.5 else rng.uniform(0, 1, 5)
        wm, wp = oracle_mod.face_values(recon, w)
        lo, hi = min(w[1], w[2], w[3]), max(w[1], w[2], w[3])
        assert lo - 1e-15 <= wm <= hi + 1e-15 and lo - 1e-15 <= wp <= hi + 1e-15
        if (w[3] - w[2]) * (w[2] - w[1]) <= 0:
            assert wm == w[2] and wp == w[2]
        # the parabola through (wm, w, wp) has no interior extremum
        if recon == PPM:
            d, w6 = wp - wm, 6 * (w[2] - 0.5 * (wm + wp))
            assert abs(w6) <= abs(d) * (1 + 1e-12) + 1e-15


def _eig(rho, vn, p, gamma):
    c = math.sqrt(gamma * p / rho)
    R = np.array([[1, -c / rho, 0, 0, c * c], [1, 0, 0, 0, 0], [0, 0, 1, 0, 0], [0, 0, 0, 1, 0],
                  [1, c / rho, 0, 0, c * c]], dtype=float)
    lam = np.array([vn - c, vn, vn, vn, vn + c])
    return lam, R


@pytest.mark.parametrize("recon", [PLM, PPM])
def test_tracing_with_zero_dt_returns_untraced(oracle_mod, recon):
    W = np.array([1.0, 0.3, -0.2, 0.1, 0.8])
    wm, wp = W - np.array([0.05, 0.01, 0.02, -0.01, 0.03]), W + np.array([0.04, 0.01, 0.02, -0.01, 0.03])
    tm, tp = oracle_mod.trace_cell(recon, 1.4, W, wm, wp, 0.0)
    assert np.array_equal(tm, wm) and np.array_equal(tp, wp)


@pytest.mark.parametrize("recon", [PLM, PPM])
@pytest.mark.parametrize("vn", [0.3, -0.3, 2.5, -2.5])
def test_single_wave_tracing_is_domain_of_dependence_average(oracle_mod, recon, vn):
    """If the in-cell profile varies along ONE eigenvector r_a, the traced face state must be the
    average of that profile over the wave's domain of dependence [face - lambda_a dt, face]
    (Colella & Woodward 1984 eq. 1.12; Colella 1990) -- computed here by direct quadrature."""
    gamma, lam_r = 5.0 / 3.0, 0.4
    W = np.array([1.3, vn, 0.2, -0.1, 0.9])
    lam, R = _eig(W[0], vn, W[4], gamma)
    for a in range(5):
        r = R[a]
        if recon == PLM:
            slope, curv = 0.02, 0.0
        else:
            slope, curv = 0.02, 0.006
        # profile W(xi) = W + r * (slope*(xi-1/2) + curv*((xi-1/2)^2 - 1/12)), xi in [0,1]; mean = W
        prof = lambda xi: slope * (xi - 0.5) + curv * ((xi - 0.5) ** 2 - 1.0 / 12.0)
        wm, wp = W + r * prof(0.0), W + r * prof(1.0)
        tm, tp = oracle_mod.trace_cell(recon, gamma, W, wm, wp, lam_r)
        y = lam[a] * lam_r

        def mean(x0, x1):
            xs = np.linspace(x0, x1, 20001)
            return np.trapezoid(prof(xs), xs) / (x1 - x0)

        # A wave that does not move toward a face stays averaged over the reference domain (that of
        # the fastest wave toward that face), as in Colella & Woodward's reference-state form.
        yp = y if y > 0 else max(lam[4] * lam_r, 0.0)
        ym = -y if y < 0 else max(-lam[0] * lam_r, 0.0)
        exp_p = W + r * (mean(1.0 - yp, 1.0) if yp > 0 else prof(1.0))
        exp_m = W + r * (mean(0.0, ym) if ym > 0 else prof(0.0))
        assert np.allclose(tp, exp_p, atol=1e-10), (a, tp, exp_p)
        assert np.allclose(tm, exp_m, atol=1e-10), (a, tm, exp_m)


def _eig_lr(rho, cs):
    """Left (rows) and right (columns) eigenvectors of the primitive-variable Euler system along n, written out from
    the literature (e.g. Stone et al. 2008, appendix A) -- independent of the oracle's project / add_wave."""
    L = np.array([[0, -rho / (2 * cs), 0, 0, 1 / (2 * cs * cs)],
                  [1, 0, 0, 0, -1 / (cs * cs)],
                  [0, 0, 1, 0, 0],
                  [0, 0, 0, 1, 0],
                  [0, rho / (2 * cs), 0, 0, 1 / (2 * cs * cs)]])
    R = np.array([[1, 1, 0, 0, 1],
                  [-cs / rho, 0, 0, 0, cs / rho],
                  [0, 0, 1, 0, 0],
                  [0, 0, 0, 1, 0],
                  [cs * cs, 0, 0, 0, cs * cs]])
    return L, R


def test_characteristic_limiting_is_R_minmod_L(oracle_mod):
    """Reading R22 (Stone et al. 2008 sect. 4.2.1): slope = R . limiter(L . dW_left, L . dW_right) with the
    eigenvectors of the cell itself.  Pins: L R = 1; random data against the matrix formula; linear data are kept
    exactly; a jump carried by one wave only (a contact: only rho differs) is limited like the scalar; and a case
    where every primitive difference keeps its sign but one characteristic amplitude changes sign, so that the
    primitive- and characteristic-limited slopes differ."""
    g = 1.4
    rng = np.random.default_rng(8)
    for _ in range(50):
        Wc = np.array([rng.uniform(0.2, 3), *rng.normal(size=3), rng.uniform(0.2, 3)])
        Wl = Wc + 0.2 * rng.normal(size=5) * np.array([0.2, 1, 1, 1, 0.2])
        Wr = Wc + 0.2 * rng.normal(size=5) * np.array([0.2, 1, 1, 1, 0.2])
        cs = math.sqrt(g * Wc[4] / Wc[0])
        L, R = _eig_lr(Wc[0], cs)
        assert np.abs(L @ R - np.eye(5)).max() < 1e-14
        aL, aR = L @ (Wc - Wl), L @ (Wr - Wc)
        lim = np.array([oracle_mod.limited_slope(oracle_mod.GMINMOD, 1.0, a, b) for a, b in zip(aL, aR)])
        got = oracle_mod.char_slope(Wl, Wc, Wr, g)
        assert np.abs(got - R @ lim).max() <= 1e-13 * (np.abs(R @ lim).max() + 1.0)
    Wc = np.array([1.3, 0.4, -0.2, 0.7, 2.1])
    d = np.array([0.05, -0.02, 0.03, 0.01, 0.08])
    assert np.abs(oracle_mod.char_slope(Wc - d, Wc, Wc + d, g) - d).max() <= 1e-15          # linear data
    sl = oracle_mod.char_slope(Wc - np.array([0.3, 0, 0, 0, 0]), Wc, Wc + np.array([0.1, 0, 0, 0, 0]), g)
    assert np.allclose(sl, [0.1, 0, 0, 0, 0], atol=1e-16)                                   # contact only
    # all primitive differences positive on both sides, but the (v - c) amplitude changes sign
    cs = math.sqrt(g * Wc[4] / Wc[0])
    dl = np.array([0.10, 0.30, 0.0, 0.0, 0.10])
    dr = np.array([0.10, 0.02, 0.0, 0.0, 0.10])
    L, R = _eig_lr(Wc[0], cs)
    assert (L @ dl)[0] * (L @ dr)[0] < 0 and (dl[[0, 1, 4]] > 0).all() and (dr[[0, 1, 4]] > 0).all()
    ch = oracle_mod.char_slope(Wc - dl, Wc, Wc + dr, g)
    pr = np.array([oracle_mod.limited_slope(oracle_mod.GMINMOD, 1.0, a, b) for a, b in zip(dl, dr)])
    assert np.abs(ch - pr).max() > 1e-3
    assert abs((L @ ch)[0]) <= 1e-15                                                         # that wave got no slope


def test_ppm_monotonisation_overshoot_branches_hand_computed(oracle_mod):
    """Colella & Woodward (1984) eq. 1.10, the two overshoot branches, on steep monotone data worked out by hand
    (PAPER.md L94 names PPM after that paper; R5: limited slopes with theta = 2, no steepening / flattening).

    Cell values a = (0, 0, 1/10, 1, 1), centre a_j = 1/10:
      slopes (gen. minmod, theta = 2; CW84 eq. 1.8): da_{j-1} = 0 (left difference is 0), da_{j+1} = 0,
        da_j = min(2*(1/10), |1 - 0|/2, 2*(9/10)) = 1/5;
      interface values (eq. 1.6): a_{j-1/2} = (0 + 1/10)/2 - (1/5 - 0)/6 = 1/20 - 1/30 = 1/60,
                                  a_{j+1/2} = (1/10 + 1)/2 - (0 - 1/5)/6 = 11/20 + 1/30 = 7/12;
      (a_R - a)(a - a_L) = (29/60)(1/12) > 0, so the cell is not an extremum;
      D = a_R - a_L = 17/30, C = a - (a_L + a_R)/2 = 1/10 - 3/10 = -1/5:  D*C = -17/150 < -D^2/6 = -289/5400,
      third line of eq. 1.10:  a_R <- 3a - 2a_L = 3/10 - 1/30 = 4/15.    Result (1/60, 4/15).
    The mirrored data (1, 1, 1/10, 0, 0) take the second line of eq. 1.10 (D*C = +17/150 > D^2/6):
      a_L <- 3a - 2a_R = 4/15, a_R = 1/60.
    Cell values (0, 0, 9/10, 1, 1): da_j = min(9/5, 1/2, 1/5) = 1/5, a_L = 9/20 - 1/30 = 5/12,
      a_R = 19/20 + 1/30 = 59/60, D = 17/30, C = 9/10 - 7/10 = 1/5, D*C = 17/150 > D^2/6:
      a_L <- 3a - 2a_R = 27/10 - 59/30 = 11/15.                       Result (11/15, 59/60); mirror (59/60, 11/15).
    A formula such as 2a - a_R in place of 3a - 2a_R (which also removes the overshoot and keeps |a_6| <= |a_R - a_L|)
    gives 11/60 / 49/60 here and fails."""
    from fractions import Fraction as Fr
    cases = [((0, 0, Fr(1, 10), 1, 1), (Fr(1, 60), Fr(4, 15))),
             ((1, 1, Fr(1, 10), 0, 0), (Fr(4, 15), Fr(1, 60))),
             ((0, 0, Fr(9, 10), 1, 1), (Fr(11, 15), Fr(59, 60))),
             ((1, 1, Fr(9, 10), 0, 0), (Fr(59, 60), Fr(11, 15)))]
    for w, (em, ep) in cases:
        wm, wp = oracle_mod.face_values(PPM, np.array([float(x) for x in w]))
        assert abs(wm - float(em)) <= 1e-15 and abs(wp - float(ep)) <= 1e-15, (w, wm, wp)
        # the monotonised parabola touches zero slope exactly at the far edge: |a_6| = |a_R - a_L|
        assert abs(abs(6 * (float(w[2]) - 0.5 * (wm + wp))) - abs(wp - wm)) <= 1e-15
    # shifted and scaled copies of the first case (the operation is affine-equivariant)
    for shift, scale in ((2.5, 1.0), (-1.0, 3.0), (0.25, -2.0)):
        w = np.array([shift + scale * float(x) for x in cases[0][0]])
        wm, wp = oracle_mod.face_values(PPM, w)
        assert wm == pytest.approx(shift + scale / 60.0, abs=4e-15) and wp == pytest.approx(shift + scale * 4.0 / 15.0, abs=4e-15)


@pytest.mark.parametrize("scheme", [1, 2])
def test_ppm_overshoot_branches_in_the_characteristic_limited_step(oracle_mod, scheme):
    """The step keeps a second copy of the PPM monotonisation for slopes limited in characteristic variables
    (R22).  On a pure contact (uniform velocity and pressure) the characteristic amplitudes of a density
    jump are (0, d rho, 0, 0, 0), so that copy must reproduce the primitive-variable face values, which the test above
    pins -- on data made of the hand-computed steep steps, so that both overshoot branches are taken.  Reference:
    the 1-D closed forms of tests/test_oracle_step.py (CTU: average over the domain of dependence; MHM: Hancock half
    step), built from oracle.face_values."""
    import torch
    from helpers import oracle_step
    from paper_1712_07070_b200 import inputs
    n = 32
    rho1 = np.full(n, 1.0)
    rho1[4:9] = 1.0 + np.array([0.0, 0.0, 0.1, 1.0, 1.0])      # the four hand-computed patterns, on a pedestal of 1
    rho1[9:12] = 2.0
    rho1[12:17] = 1.0 + np.array([1.0, 1.0, 0.1, 0.0, 0.0])
    rho1[20:25] = 1.0 + np.array([0.0, 0.0, 0.9, 1.0, 1.0])
    rho1[25:27] = 2.0
    rho1[27:32] = 1.0 + np.array([1.0, 1.0, 0.9, 0.0, 0.0])
    rho = torch.from_numpy(rho1)[None, None, :].expand(16, 16, n).contiguous()
    one = torch.ones_like(rho)
    v = 0.7
    f = inputs.prim_to_cons(rho, v * one, 0 * one, 0 * one, one, 1.4)
    dh, dt = 1.0 / n, 0.4 / n
    nu = v * dt / dh
    new, _ = oracle_step(oracle_mod, f, dt, dh, 1.4, scheme, PPM, 2, opts=oracle_mod.make_opts(char_limiting=True))
    face, hit = np.empty(n), 0
    for i in range(n):
        w5 = np.array([rho1[(i + m) % n] for m in range(-2, 3)])
        wm, wp = oracle_mod.face_values(PPM, w5)
        d, w6 = wp - wm, 6 * (rho1[i] - 0.5 * (wm + wp))
        hit += abs(abs(w6) - abs(d)) < 1e-14 and abs(d) > 0.1
        if scheme == 2:      # CTU: average of the parabola over [x_f - v dt, x_f]
            face[i] = wp - 0.5 * nu * (d - (1 - 2.0 / 3.0 * nu) * w6)
        else:                # MHM: face value minus half the flux difference across the cell
            face[i] = wp - 0.5 * nu * d
    assert hit >= 4                                           # the overshoot branches were taken
    ref = rho1 - nu * (face - np.roll(face, 1))
    assert np.abs(new[0, 2, 7].numpy() - ref).max() <= 5e-14
