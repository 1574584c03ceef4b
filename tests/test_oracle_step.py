"""Whole-step pins of the oracle (oracle/hydro_oracle.c): invariants and special cases that the
paper and the mathematics fix.  CPU only."""
import itertools
import math

import numpy as np
import pytest
import torch

from helpers import oracle_run, oracle_step
from paper_1712_07070_b200 import inputs

MHM, CTU, VL = 1, 2, 3
PLM, PPM = 1, 2
ROE, HLLC, HLLE = 1, 2, 3
EXACT = 4
COMBOS = list(itertools.product((MHM, CTU), (PLM, PPM), (ROE, HLLC, HLLE))) + [(MHM, PLM, EXACT), (CTU, PPM, EXACT)] + \
    [(VL, PLM, ROE), (VL, PLM, HLLC), (VL, PLM, HLLE)]
G53 = 5.0 / 3.0


def _turb(n=32, seed=1712, mach=1.0, entropy=False):
    return inputs.turbulence_field(n, seed, kmax=4, gamma=G53, mach=mach, entropy=entropy)


def _dt(oracle, field, dh, gamma, cfl, scheme, opts=None):
    u = inputs.interior(inputs.pack_periodic(field)).contiguous().numpy()
    return oracle.cfl_dt(u, dh, gamma, cfl, scheme, opts)[0]


@pytest.mark.parametrize("scheme,recon,solver", COMBOS)
def test_conservation_on_periodic_box(oracle_mod, scheme, recon, solver):
    """conservation to machine precision (pure hydro, closed domain)."""
    f = _turb()
    dh = 1.0 / 32
    dt = _dt(oracle_mod, f, dh, G53, 0.4, scheme)
    new, r = oracle_step(oracle_mod, f, dt, dh, G53, scheme, recon, solver)
    assert r["stats"]["n_unphysical"] == 0
    for v in range(5):
        s0, s1 = math.fsum(f[v].flatten().tolist()), math.fsum(new[v].flatten().tolist())
        scale = math.fsum(f[v].abs().flatten().tolist()) + 1.0
        assert abs(s1 - s0) <= 1e-13 * scale, (v, s0, s1)
    assert (new - f).abs().max() > 1e-3       # and something did happen


@pytest.mark.parametrize("scheme,recon,solver", [(MHM, PLM, ROE), (CTU, PPM, HLLC), (MHM, PPM, HLLE), (VL, PLM, ROE)])
def test_boundary_fluxes_of_neighbouring_groups_are_bitwise_equal(oracle_mod, scheme, recon, solver):
    """the flux through a face shared by two groups is computed twice and must agree
    bit for bit; also the mid-plane (p=1) equals the difference form of the update."""
    f = _turb()
    dh = 1.0 / 32
    dt = _dt(oracle_mod, f, dh, G53, 0.4, scheme)
    _, r = oracle_step(oracle_mod, f, dt, dh, G53, scheme, recon, solver)
    fl = r["flux"].reshape(2, 2, 2, 3, 3, 5, 16, 16)      # [gz,gy,gx,axis,plane,...]
    for gz, gy, gx in itertools.product(range(2), repeat=3):
        assert np.array_equal(fl[gz, gy, gx, 0, 2], fl[gz, gy, (gx + 1) % 2, 0, 0])
        assert np.array_equal(fl[gz, gy, gx, 1, 2], fl[gz, (gy + 1) % 2, gx, 1, 0])
        assert np.array_equal(fl[gz, gy, gx, 2, 2], fl[(gz + 1) % 2, gy, gx, 2, 0])


@pytest.mark.parametrize("scheme,recon,solver", [(MHM, PLM, HLLE), (CTU, PLM, ROE), (VL, PLM, HLLC)])
def test_flux_out_reproduces_update_of_a_boundary_slab(oracle_mod, scheme, recon, solver):
    """Sum over a half-group slab: d(sum U)/dt = -(flux through its faces)/dh.  With periodic y,z
    sums over a whole x-slab [0,8) of the 32^3 box, only the x-planes 0 and 8 contribute."""
    f = _turb()
    dh = 1.0 / 32
    dt = _dt(oracle_mod, f, dh, G53, 0.4, scheme)
    new, r = oracle_step(oracle_mod, f, dt, dh, G53, scheme, recon, solver)
    fl = r["flux"].reshape(2, 2, 2, 3, 3, 5, 16, 16)
    for v in range(5):
        dsum = (new[v, :, :, 0:8] - f[v, :, :, 0:8]).sum().item()
        fin = fl[:, :, 0, 0, 0, v].sum()       # x-plane 0 of the gx=0 groups
        fout = fl[:, :, 0, 0, 1, v].sum()      # x-plane 8
        assert dsum == pytest.approx(-(dt / dh) * (fout - fin), rel=1e-9, abs=1e-11)


@pytest.mark.parametrize("scheme,recon,solver", COMBOS)
def test_uniform_state_is_bitwise_invariant(oracle_mod, scheme, recon, solver):
    n = 16
    one = torch.ones((n, n, n), dtype=torch.float64)
    f = inputs.prim_to_cons(1.3 * one, 0.7 * one, -0.45 * one, 0.3 * one, 0.9 * one, G53)
    new, _ = oracle_step(oracle_mod, f, 0.01, 1.0 / n, G53, scheme, recon, solver)
    assert torch.equal(new, f)


@pytest.mark.parametrize("scheme,recon,solver", COMBOS)
def test_cyclic_permutation_symmetry(oracle_mod, scheme, recon, solver):
    """Relabel the axes (x,y,z) -> (y,z,x): the solver must commute with it (<= 1e-13: the three-term
    sums re-associate, so not bitwise)."""
    f = _turb(seed=99)
    dh, dt = 1.0 / 32, 0.004
    new, _ = oracle_step(oracle_mod, f, dt, dh, G53, scheme, recon, solver)
    # P: array [z,y,x] -> [x,z,y] i.e. the old x axis becomes the new z axis, old z -> new y, old y -> new x
    def P(a):
        b = a.permute(0, 3, 1, 2).contiguous()
        # momentum: new (mx', my', mz') = components along new axes = old (my, mz, mx)
        return torch.stack([b[0], b[2], b[3], b[1], b[4]], dim=0)
    newP, _ = oracle_step(oracle_mod, P(f), dt, dh, G53, scheme, recon, solver)
    ref = P(new)
    assert (newP - ref).abs().max().item() <= 1e-13 * ref.abs().max().item()


@pytest.mark.parametrize("scheme,recon,solver", [(MHM, PLM, ROE), (CTU, PPM, HLLC), (CTU, PLM, HLLE), (MHM, PPM, HLLC), (VL, PLM, HLLE)])
def test_mirror_symmetry(oracle_mod, scheme, recon, solver):
    f = _turb(seed=5)
    dh, dt = 1.0 / 32, 0.004
    new, _ = oracle_step(oracle_mod, f, dt, dh, G53, scheme, recon, solver)
    def M(a):
        b = torch.flip(a, dims=[3]).clone()
        b[1] = -b[1]
        return b
    newM, _ = oracle_step(oracle_mod, M(f), dt, dh, G53, scheme, recon, solver)
    assert (newM - M(new)).abs().max().item() <= 1e-13 * new.abs().max().item()


@pytest.mark.parametrize("scheme,recon,solver", COMBOS)
def test_one_dimensional_data_stay_one_dimensional_bitwise(oracle_mod, scheme, recon, solver):
    f = inputs.sod_field(32, 1.4)
    new, _ = oracle_step(oracle_mod, f, 0.2 / 32, 1.0 / 32, 1.4, scheme, recon, solver)
    assert torch.equal(new, new[:, :1, :1, :].expand_as(new))
    assert new[2].abs().max() == 0 and new[3].abs().max() == 0


def _minmod(a, b):
    return np.where(a * b > 0, np.sign(a) * np.minimum(np.abs(a), np.abs(b)), 0.0)


@pytest.mark.parametrize("scheme,solver", [(MHM, ROE), (MHM, HLLC), (CTU, ROE), (CTU, HLLC)])
def test_contact_advection_reduces_to_second_order_upwind_advection(oracle_mod, scheme, solver):
    """Uniform v and P, varying rho: the Euler system reduces to linear advection of rho.  Roe and
    HLLC resolve a moving contact exactly, so MHM+PLM (and CTU+PLM in 1-D) must equal the textbook
    second-order upwind (MUSCL/Fromm-type) scheme  rho_i - nu (r_{i+1/2} - r_{i-1/2}),
    r_{i+1/2} = rho_i + (1-nu)/2 * minmod slope   (Toro 2009 sect. 13.4; van Leer 1979)."""
    n = 32
    x = (np.arange(n) + 0.5) / n
    rho1 = 1.0 + 0.3 * np.sin(2 * np.pi * x) + 0.2 * (np.abs(x - 0.5) < 0.2)
    rho = torch.from_numpy(rho1)[None, None, :].expand(16, 16, n).contiguous()
    one = torch.ones_like(rho)
    v = 0.8
    f = inputs.prim_to_cons(rho, v * one, 0 * one, 0 * one, one, 1.4)
    dh, dt = 1.0 / n, 0.3 / n / v * 1.0
    nu = v * dt / dh
    new, _ = oracle_step(oracle_mod, f, dt, dh, 1.4, scheme, PLM, solver)
    s = _minmod(rho1 - np.roll(rho1, 1), np.roll(rho1, -1) - rho1)
    face = rho1 + 0.5 * (1 - nu) * s
    ref = rho1 - nu * (face - np.roll(face, 1))
    assert np.abs(new[0, 3, 5].numpy() - ref).max() <= 2e-14
    # velocity and pressure stay uniform
    assert np.abs(new[1, 3, 5].numpy() / new[0, 3, 5].numpy() - v).max() <= 1e-13


def test_mhm_three_d_contact_advection_closed_form(oracle_mod):
    """Same reduction in 3-D for the unsplit MUSCL-Hancock scheme: the half-step predictor adds
    -(1/2) sum_d nu_d slope_d to every face value (Toro 2009 sect. 16.5)."""
    n = 16
    f0 = inputs.blob_field(n, G53, v=(0.9, -0.6, 0.4))
    rho = f0[0].numpy()
    vel = (0.9, -0.6, 0.4)
    dh, dt = 1.0 / n, 0.25 / n
    new, _ = oracle_step(oracle_mod, f0, dt, dh, G53, MHM, PLM, HLLC)
    ax = {0: 2, 1: 1, 2: 0}      # direction -> array axis
    slopes = {d: _minmod(rho - np.roll(rho, 1, ax[d]), np.roll(rho, -1, ax[d]) - rho) for d in range(3)}
    half = -0.5 * sum(vel[d] * dt / dh * slopes[d] for d in range(3))
    ref = rho.copy()
    for d in range(3):
        nu = vel[d] * dt / dh
        if vel[d] > 0:
            face = rho + 0.5 * slopes[d] + half                 # value at i+1/2 from cell i
            ref -= nu * (face - np.roll(face, 1, ax[d]))
        else:
            face = rho - 0.5 * slopes[d] + half                 # value at i-1/2 from cell i
            ref -= nu * (np.roll(face, -1, ax[d]) - face)
    assert np.abs(new[0].numpy() - ref).max() <= 5e-14


@pytest.mark.parametrize("recon", [PLM, PPM])
def test_ctu_one_d_contact_advection_uses_domain_of_dependence_average(oracle_mod, recon):
    """CTU in 1-D: the face value is the average of the reconstructed profile over [x_f - v dt, x_f]
    (Colella 1990).  For PPM the profile is the monotonised parabola, integrated here in closed form
    from the oracle's own (separately pinned) face values."""
    n = 32
    x = (np.arange(n) + 0.5) / n
    rho1 = 1.0 + 0.3 * np.sin(2 * np.pi * x) + 0.1 * np.sin(6 * np.pi * x)
    rho = torch.from_numpy(rho1)[None, None, :].expand(16, 16, n).contiguous()
    one = torch.ones_like(rho)
    v = 0.7
    f = inputs.prim_to_cons(rho, v * one, 0 * one, 0 * one, one, 1.4)
    dh, dt = 1.0 / n, 0.4 / n
    nu = v * dt / dh
    new, _ = oracle_step(oracle_mod, f, dt, dh, 1.4, CTU, recon, HLLC)
    face = np.empty(n)
    for i in range(n):
        w5 = np.array([rho1[(i + m) % n] for m in range(-2, 3)])
        wm, wp = oracle_mod.face_values(recon, w5)
        d, w6 = wp - wm, (6 * (rho1[i] - 0.5 * (wm + wp)) if recon == PPM else 0.0)
        face[i] = wp - 0.5 * nu * (d - (1 - 2.0 / 3.0 * nu) * w6)
    ref = rho1 - nu * (face - np.roll(face, 1))
    assert np.abs(new[0, 2, 7].numpy() - ref).max() <= 2e-14


@pytest.mark.parametrize("scheme,recon,solver", COMBOS)
def test_sod_converges_to_exact_solution(oracle_mod, scheme, recon, solver):
    """BASELINE.json config 1 data; exact solution from Toro's iterative procedure (tests/exact_riemann.py,
    itself pinned to the printed values in tests/golden/sod_exact.txt).  The periodic wrap adds a
    mirrored tube at x=0; until t=0.12 the two wave fans do not meet."""
    import exact_riemann as er
    t_end, gamma = 0.12, 1.4
    errs = []
    for n in (64, 128):
        f = inputs.sod_field(n, gamma, nyz=16)
        cfl = 0.4 if scheme == CTU else 0.8
        out, nsteps = oracle_run(oracle_mod, f, t_end, 1.0 / n, gamma, cfl, scheme, recon, solver)
        x = (np.arange(n) + 0.5) / n
        rho_ex = np.empty(n)
        mid = (x > 0.25) & (x < 0.75)
        rho_ex[mid] = er.sample(1, 0, 1, 0.125, 0, 0.1, gamma, (x[mid] - 0.5) / t_end)[0]
        xs = np.where(x[~mid] > 0.5, x[~mid] - 1.0, x[~mid])
        rho_ex[~mid] = er.sample(0.125, 0, 0.1, 1, 0, 1, gamma, xs / t_end)[0]
        rho = out[0, 3, 4].numpy()
        errs.append(np.abs(rho - rho_ex).mean())
        if n == 128:
            # plateaus between tail/contact and contact/shock, within 2 % at N=128
            ps, us = er.star_state(1, 0, 1, 0.125, 0, 0.1, gamma)
            xl = 0.5 + 0.5 * (-0.0702728126 + us) * t_end
            xr = 0.5 + 0.5 * (us + 1.7521557320) * t_end
            assert rho[int(xl * n)] == pytest.approx(0.4263194282, rel=0.02)
            assert rho[int(xr * n)] == pytest.approx(0.2655737117, rel=0.02)
    order = math.log(errs[0] / errs[1], 2.0)
    assert errs[1] < 1.2e-2 and order >= 0.7, (errs, order)


@pytest.mark.parametrize("scheme,recon,cfl", [(MHM, PLM, 1.0), (MHM, PPM, 1.0), (CTU, PLM, 0.5), (CTU, PPM, 0.5), (VL, PLM, 1.0)])
def test_stable_at_the_stated_cfl_limit(oracle_mod, scheme, recon, cfl):
    """CTU needs C_CFL <= 0.5, the others support C_CFL <= 1.0 (with their own Eq. 1 / 2)."""
    f = inputs.blob_field(16, G53)
    lo, hi = f[0].min().item(), f[0].max().item()
    out, n = oracle_run(oracle_mod, f, 1e9, 1.0 / 16, G53, cfl, scheme, recon, HLLC, max_steps=60)
    assert n == 60 and torch.isfinite(out).all()
    assert out[0].min().item() >= lo - 0.02 and out[0].max().item() <= hi + 0.02


@pytest.mark.parametrize("scheme,recon", [(MHM, PLM), (CTU, PLM), (MHM, PPM), (CTU, PPM), (VL, PLM)])
def test_ghost_footprint(oracle_mod, scheme, recon):
    """CTU+PPM needs 3 ghost zones.  MHM/CTU + PLM must ignore ghost layer 3; no variant's result depends on
    the triple-corner ghosts; PPM must read layer 3, and so must VL + PLM (its half-step predictor reaches one cell
    further than the reconstruction: that is why VL + PPM would need a fourth zone)."""
    f = _turb(n=16, seed=3)
    p = inputs.pack_periodic(f).numpy()
    dt, dh = 0.002, 1.0 / 16
    base = oracle_mod.fluid_advance(p, dt, dh, G53, scheme, recon, HLLC)
    q = p.copy()
    outer = np.ones((22, 22, 22), dtype=bool)
    outer[1:21, 1:21, 1:21] = False
    q[:, :, outer] *= 1.5                      # outermost ghost layer (layer 3)
    r = oracle_mod.fluid_advance(q, dt, dh, G53, scheme, recon, HLLC)
    same = np.array_equal(r["out"], base["out"]) and np.array_equal(r["flux"], base["flux"])
    assert same == (recon == PLM and scheme != VL)
    q = p.copy()
    idx = np.arange(22)
    gh = (idx < 3) | (idx >= 19)
    corner = gh[:, None, None] & gh[None, :, None] & gh[None, None, :]
    q[:, :, corner] *= 1.5
    r = oracle_mod.fluid_advance(q, dt, dh, G53, scheme, recon, HLLC)
    assert np.array_equal(r["out"], base["out"]) and np.array_equal(r["flux"], base["flux"])


def test_riemann_solves_per_cell(oracle_mod):
    """PAPER.md L90 / L521: MHM needs 3 and CTU 6 Riemann solves per cell.  Per group the final pass is
    3*17*16*16 faces (3/cell once shared faces are counted once); CTU adds the first pass on the
    faces of the cells [-1,16]^3."""
    p = inputs.pack_periodic(_turb(n=16)).numpy()
    a = oracle_mod.fluid_advance(p, 0.002, 1.0 / 16, G53, MHM, PLM, HLLC)["stats"]
    b = oracle_mod.fluid_advance(p, 0.002, 1.0 / 16, G53, CTU, PLM, HLLC)["stats"]
    assert a["n_riemann"] == a["n_riemann_final"] == 3 * 17 * 16 * 16
    assert 3 * 16 ** 3 * 16 // 17 <= 3 * 16 ** 3                      # shared faces: 16 of 17 unique
    assert b["n_riemann_final"] == 3 * 17 * 16 * 16
    assert b["n_riemann"] - b["n_riemann_final"] == 3 * 17 * 18 * 18
    # VL: 3 + 3 per cell too (first-order pass on the faces of the cells [-2,17]^3, then the final pass)
    v = oracle_mod.fluid_advance(p, 0.002, 1.0 / 16, G53, VL, PLM, HLLC)["stats"]
    assert v["n_riemann_final"] == 3 * 17 * 16 * 16
    assert v["n_riemann"] - v["n_riemann_final"] == 3 * 21 * 20 * 20


@pytest.mark.parametrize("scheme,recon,solver", [(MHM, PLM, ROE), (CTU, PPM, HLLC), (MHM, PPM, HLLE), (CTU, PLM, ROE)])
def test_characteristic_limiting_whole_step(oracle_mod, scheme, recon, solver):
    """Reading R22 in the whole step: with slopes limited in characteristic variables the step still conserves to
    round-off, commutes with the relabelling of the axes, leaves a uniform state untouched bit for bit, differs from
    the primitive-limited step, and resolves the Sod tube at least as well (L1 density error vs the exact solution)."""
    import exact_riemann as er
    opts = oracle_mod.make_opts(char_limiting=True)
    f = _turb()
    dh = 1.0 / 32
    dt = _dt(oracle_mod, f, dh, G53, 0.4, scheme)
    new, r = oracle_step(oracle_mod, f, dt, dh, G53, scheme, recon, solver, opts=opts)
    ref, _ = oracle_step(oracle_mod, f, dt, dh, G53, scheme, recon, solver)
    assert r["stats"]["n_unphysical"] == 0
    for v in range(5):
        s0, s1 = math.fsum(f[v].flatten().tolist()), math.fsum(new[v].flatten().tolist())
        assert abs(s1 - s0) <= 1e-13 * (math.fsum(f[v].abs().flatten().tolist()) + 1.0)
    assert (new - ref).abs().max().item() <= 1e-12      # on this smooth field both limiters pick the same side everywhere

    def P(a):
        b = a.permute(0, 3, 1, 2).contiguous()
        return torch.stack([b[0], b[2], b[3], b[1], b[4]], dim=0)
    newP, _ = oracle_step(oracle_mod, P(f), dt, dh, G53, scheme, recon, solver, opts=opts)
    assert (newP - P(new)).abs().max().item() <= 1e-13 * new.abs().max().item()
    uni = torch.ones_like(f) * torch.tensor([1.3, 0.4, -0.7, 0.2, 3.1])[:, None, None, None]
    u1, _ = oracle_step(oracle_mod, uni, dt, dh, G53, scheme, recon, solver, opts=opts)
    assert torch.equal(u1, uni)
    # Sod tube, 128 cells, t = 0.1
    n, gamma = 128, 1.4
    errs, finals = [], []
    for o in (None, oracle_mod.make_opts(char_limiting=True)):
        u = inputs.sod_field(n, gamma, nyz=16)
        t = 0.0
        while t < 0.1 - 1e-12:
            dts = min(_dt(oracle_mod, u, 1.0 / n, gamma, 0.4, scheme), 0.1 - t)
            u, _ = oracle_step(oracle_mod, u, dts, 1.0 / n, gamma, scheme, recon, solver, opts=o)
            t += dts
        x = (np.arange(n) + 0.5) / n
        rho_e = er.sample(1, 0, 1, 0.125, 0, 0.1, gamma, (x[16:112] - 0.5) / 0.1)[0]      # away from the periodic image
        errs.append(np.abs(u[0, 0, 0, 16:112].numpy() - rho_e).mean())
        finals.append(u)
    assert errs[1] <= 1.1 * errs[0], errs
    assert (finals[0] - finals[1]).abs().max().item() > 1e-4      # at the waves of the tube the two limiters do differ


# ---------------------------------------------------------------------------------------------------------------
# Pins of the CTU transverse flux-gradient correction (oracle step O4-CTU (c); "6 Riemann solvers per
# cell per time-step, similar to ATHENA", L168 C_CFL <= 0.5; R7).  A 1-D test cannot see this step (the
# transverse flux differences vanish), so the three tests below use data with gradients in all directions.
# ---------------------------------------------------------------------------------------------------------------
def _ctu_plm_contact_reference(rho, vel, lam_r):
    """The 6-solve CTU scheme written out for linear advection of rho (uniform velocity and pressure; Roe and HLLC
    resolve a moving contact exactly, i.e. every Riemann flux is v_d times the upwind face density):
      traced face value of cell c along d (PLM, Colella 1990):  rho_c +- 1/2 (1 -+ nu_d) s_d  on the downwind (+ for
        v_d > 0, - for v_d < 0) face, nu_d = v_d dt/dh, s_d the minmod slope;
      first-pass flux  F*_d(c + e_d/2) = v_d * (upwind traced value);
      the d-face states of cell c are corrected by  -1/2 dt/dh [F*_d'(c + e_d'/2) - F*_d'(c - e_d'/2)]  for BOTH
        transverse directions d' != d  (Colella 1990 eq. 2.17 ff.; Stone et al. 2008 sect. 4.2 step 5 without B);
      second pass: F_d = v_d * (upwind corrected value); update rho - dt/dh sum_d [F_d(+) - F_d(-)].
    rho: numpy [nz, ny, nx], periodic."""
    ax = {0: 2, 1: 1, 2: 0}      # direction -> array axis
    up, f1 = {}, {}
    for d in range(3):
        s = _minmod(rho - np.roll(rho, 1, ax[d]), np.roll(rho, -1, ax[d]) - rho)
        nu = vel[d] * lam_r
        # upwind traced value, stored at the cell that owns it (v>0: its + face, v<0: its - face)
        up[d] = rho + 0.5 * (1.0 - nu) * s if vel[d] > 0 else rho - 0.5 * (1.0 + nu) * s
        # first-pass flux at face c + e_d/2
        f1[d] = vel[d] * (up[d] if vel[d] > 0 else np.roll(up[d], -1, ax[d]))
    new = rho.copy()
    for d in range(3):
        corr = up[d].copy()
        for dp in range(3):
            if dp != d:
                corr -= 0.5 * lam_r * (f1[dp] - np.roll(f1[dp], 1, ax[dp]))
        flux = vel[d] * (corr if vel[d] > 0 else np.roll(corr, -1, ax[d]))      # at face c + e_d/2
        new -= lam_r * (flux - np.roll(flux, 1, ax[d]))
    return new


@pytest.mark.parametrize("solver", [ROE, HLLC])
@pytest.mark.parametrize("vel", [(0.9, -0.6, 0.4), (-0.5, 0.8, -0.7), (0.3, 0.45, 0.6), (-0.85, -0.2, -0.5)])
def test_ctu_three_d_contact_advection_closed_form(oracle_mod, solver, vel):
    """CTU + PLM on an obliquely advected density field (all three velocity components non-zero, mixed signs):
    the result must equal the corner-transport-upwind scheme for linear advection written out above, to round-off.
    Kills: a missing transverse correction, a wrong coefficient (e.g. 1 and 0 instead of 1/2 and 1/2), a correction
    built from the wrong faces or the wrong transverse directions, a wrong sign."""
    n = 16
    z, y, x = np.meshgrid(*(((np.arange(n) + 0.5) / n,) * 3), indexing="ij")
    rho = (1.0 + 0.4 * np.sin(2 * np.pi * x) * np.cos(2 * np.pi * y) + 0.25 * np.cos(2 * np.pi * (y - 2 * z))
           + 0.3 * (np.abs(x - 0.5) + np.abs(y - 0.4) + np.abs(z - 0.6) < 0.45))      # smooth part + a step
    t = torch.from_numpy(rho)
    one = torch.ones_like(t)
    f0 = inputs.prim_to_cons(t, vel[0] * one, vel[1] * one, vel[2] * one, one.clone(), G53)
    dh, dt = 1.0 / n, 0.3 / n
    new, r = oracle_step(oracle_mod, f0, dt, dh, G53, CTU, PLM, solver)
    assert r["stats"]["n_pred_revert"] == 0 and r["stats"]["n_roe_fallback"] == 0
    ref = _ctu_plm_contact_reference(rho, vel, dt / dh)
    assert np.abs(new[0].numpy() - ref).max() <= 5e-14
    # the transverse terms are not small here: without them the result is off by far more than the tolerance
    unc = rho.copy()
    for d, a in ((0, 2), (1, 1), (2, 0)):
        s = _minmod(rho - np.roll(rho, 1, a), np.roll(rho, -1, a) - rho)
        nu = vel[d] * dt / dh
        face = rho + 0.5 * (1 - nu) * s if vel[d] > 0 else np.roll(rho - 0.5 * (1 + nu) * s, -1, a)
        unc -= nu * (face - np.roll(face, 1, a))
    assert np.abs(unc - ref).max() > 1e-3
    # velocity and pressure stay uniform
    w = new.numpy()
    for d in range(3):
        assert np.abs(w[1 + d] / w[0] - vel[d]).max() <= 1e-13
    pres = (G53 - 1.0) * (w[4] - 0.5 * (w[1] ** 2 + w[2] ** 2 + w[3] ** 2) / w[0])
    assert np.abs(pres - 1.0).max() <= 1e-13


def _ctu_cell_from_building_blocks(o, p, cell, lam_r, gamma, recon, solver):
    """The CTU update of ONE cell of a padded group rebuilt from the oracle's separately pinned building blocks
    (face_values, trace_cell, riemann -- tests/test_oracle_recon.py, test_oracle_riemann.py) with the wiring of the
    6-solve scheme (Stone et al. 2008 sect. 4.2 without magnetic field) written independently here:
      (a) traced primitive states of a cell along d;  (b) F*_d at face c + e_d/2 from the + state of c and the - state
      of c + e_d;  (c) d-face states of c, in conserved variables, minus dt/(2 dh) times the flux differences across c
      in the two other directions;  (d) final fluxes from the corrected states;  U - dt/dh sum_d dF_d.
    p: [5, 22, 22, 22] numpy; cell = (i, j, k) padded indices."""
    gm1 = gamma - 1.0
    step = {0: (1, 0, 0), 1: (0, 1, 0), 2: (0, 0, 1)}

    def prim(c):
        U = p[:, c[2], c[1], c[0]]
        v = U[1:4] / U[0]
        return np.array([U[0], v[0], v[1], v[2], gm1 * (U[4] - 0.5 * U[0] * (v ** 2).sum())])

    def cons(W):
        return np.array([W[0], W[0] * W[1], W[0] * W[2], W[0] * W[3],
                         W[4] / gm1 + 0.5 * W[0] * (W[1] ** 2 + W[2] ** 2 + W[3] ** 2)])

    def shift(c, d, m):
        return tuple(c[a] + m * step[d][a] for a in range(3))

    traced_memo, f1_memo = {}, {}

    def traced(c, d):
        """conserved (minus, plus) traced states of cell c along d"""
        if (c, d) not in traced_memo:
            rot = [0, 1 + d, 1 + (d + 1) % 3, 1 + (d + 2) % 3, 4]
            strip = np.array([prim(shift(c, d, m)) for m in range(-2, 3)])      # [5 cells, 5 vars]
            wm, wp = np.empty(5), np.empty(5)
            for v in range(5):
                wm[v], wp[v] = o.face_values(recon, strip[:, v])
            tm, tp = o.trace_cell(recon, gamma, strip[2][rot], wm[rot], wp[rot], lam_r)
            Tm, Tp = np.empty(5), np.empty(5)
            Tm[rot], Tp[rot] = tm, tp
            traced_memo[(c, d)] = (cons(Tm), cons(Tp))
        return traced_memo[(c, d)]

    def f1(c, d):
        """first-pass flux at face c + e_d/2"""
        if (c, d) not in f1_memo:
            f1_memo[(c, d)] = o.riemann(solver, d, traced(c, d)[1], traced(shift(c, d, 1), d)[0], gamma)[0]
        return f1_memo[(c, d)]

    def corrected(c, d, side):
        U = traced(c, d)[side].copy()
        for dp in range(3):
            if dp != d:
                U -= 0.5 * lam_r * (f1(c, dp) - f1(shift(c, dp, -1), dp))
        return U

    def f2(c, d):
        return o.riemann(solver, d, corrected(c, d, 1), corrected(shift(c, d, 1), d, 0), gamma)[0]

    U = p[:, cell[2], cell[1], cell[0]].copy()
    for d in range(3):
        U -= lam_r * (f2(cell, d) - f2(shift(cell, d, -1), d))
    return U


@pytest.mark.parametrize("recon,solver", [(PLM, ROE), (PPM, HLLC), (PPM, HLLE)])
def test_ctu_cell_rebuilt_from_pinned_building_blocks(oracle_mod, recon, solver):
    """General (non-contact) data: the update of sampled cells, all five variables, equals the 6-solve wiring above
    applied to the pinned building blocks.  Covers what the contact closed form cannot: the momentum and energy
    components of the transverse correction and the conserved <-> primitive conversions around it."""
    f = _turb(n=16, seed=11)
    p = inputs.pack_periodic(f).numpy()
    dh = 1.0 / 16
    dt = _dt(oracle_mod, f, dh, G53, 0.4, CTU)
    r = oracle_mod.fluid_advance(p, dt, dh, G53, CTU, recon, solver)
    assert r["stats"]["n_pred_revert"] == 0
    for (i, j, k) in ((0, 0, 0), (15, 7, 3), (8, 15, 12), (5, 9, 15)):      # corners / faces of the group: halo states used
        ref = _ctu_cell_from_building_blocks(oracle_mod, p[0], (i + 3, j + 3, k + 3), dt / dh, G53, recon, solver)
        got = r["out"][0, :, k, j, i]
        assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max(), (i, j, k, got, ref)


@pytest.mark.parametrize("recon", [PLM, PPM])
def test_ctu_diagonal_advection_is_second_order(oracle_mod, recon):
    """Smooth density wave advected along the x-y diagonal at C_CFL = 0.45 for a fixed time: the L1 error must fall
    at second order (>= 1.8 between N = 32 and 64).  Without the transverse correction the unsplit scheme lacks the
    v_x v_y d2/dxdy term of the second-order Taylor expansion in time and is first order (and, at this CFL number,
    unstable: Colella 1990 sect. 2): measured orders 1.2 (PLM) and 0.9 (PPM) with the correction removed, 2.15 / 2.04
    with it.  PLM runs with the generalized-minmod parameter theta = 2 (the plain minmod of theta = 1 clips the
    extrema of the sine wave and by itself lowers the L1 order to 1.79)."""
    vel, t_end = (1.0, 0.75, 0.0), 0.25
    opts = oracle_mod.make_opts(theta=2.0)
    errs = []
    for n in (16, 32, 64):
        x = ((np.arange(n) + 0.5) / n)[None, None, :]
        y = ((np.arange(n) + 0.5) / n)[None, :, None]
        rho_fn = lambda xx, yy: 1.0 + 0.3 * np.sin(2 * np.pi * (xx + yy)) + 0.0 * xx * yy
        rho0 = np.broadcast_to(rho_fn(x, y), (16, n, n)).copy()
        t = torch.from_numpy(rho0)
        one = torch.ones_like(t)
        f = inputs.prim_to_cons(t, vel[0] * one, vel[1] * one, 0.0 * one, one.clone(), 1.4)
        out, _ = oracle_run(oracle_mod, f, t_end, 1.0 / n, 1.4, 0.45, CTU, recon, HLLC, opts)
        exact = np.broadcast_to(rho_fn(x - vel[0] * t_end, y - vel[1] * t_end), (16, n, n))
        errs.append(np.abs(out[0].numpy() - exact).mean())
    order = math.log(errs[1] / errs[2], 2.0)
    assert order >= 1.8, (errs, order)
    assert errs[2] < 1e-3


# ---------------------------------------------------------------------------------------------------------------
# VL scheme ("a variant of the MUSCL-Hancock scheme (VL; Falle 1991; van Leer 2006)"; R26)
# ---------------------------------------------------------------------------------------------------------------
def _vl_contact_reference(rho, vel, lam_r):
    """The VL scheme written out for linear advection of rho (uniform velocity and pressure, exact upwinding by Roe /
    HLLC): first-order upwind half step  rho_h = rho - 1/2 sum_d nu_d (rho - rho_upwind-neighbour),  minmod slopes of
    rho_h, second-order upwind fluxes  v_d (rho_h +- 1/2 slope)  from the upwind cell, full step from rho.
    (van Leer 2006 sect. 5; Stone & Gardiner 2009 sect. 3 steps 1-6 without magnetic field.)"""
    ax = {0: 2, 1: 1, 2: 0}
    rh = rho.copy()
    for d in range(3):
        nu = vel[d] * lam_r
        up = np.roll(rho, 1, ax[d]) if vel[d] > 0 else np.roll(rho, -1, ax[d])
        rh -= 0.5 * abs(nu) * (rho - up)
    new = rho.copy()
    for d in range(3):
        s = _minmod(rh - np.roll(rh, 1, ax[d]), np.roll(rh, -1, ax[d]) - rh)
        face = rh + 0.5 * s if vel[d] > 0 else np.roll(rh - 0.5 * s, -1, ax[d])      # at c + e_d/2
        new -= vel[d] * lam_r * (face - np.roll(face, 1, ax[d]))
    return new


@pytest.mark.parametrize("solver", [ROE, HLLC])
@pytest.mark.parametrize("vel", [(0.9, -0.6, 0.4), (-0.5, 0.8, -0.7), (0.8, 0.0, 0.0)])
def test_vl_contact_advection_closed_form(oracle_mod, solver, vel):
    """1-D (third velocity) and oblique 3-D contact advection: VL + PLM equals the scheme above to round-off.
    Kills: a predictor over dt instead of dt/2, slopes taken from U^n instead of the half-step state, a final update
    from the half-step state instead of U^n, Hancock-type evolution left in, wrong upwind side."""
    n = 16
    z, y, x = np.meshgrid(*(((np.arange(n) + 0.5) / n,) * 3), indexing="ij")
    rho = (1.0 + 0.4 * np.sin(2 * np.pi * x) * np.cos(2 * np.pi * y) + 0.25 * np.cos(2 * np.pi * (y - 2 * z))
           + 0.3 * (np.abs(x - 0.5) + np.abs(y - 0.4) + np.abs(z - 0.6) < 0.45))
    t = torch.from_numpy(rho)
    one = torch.ones_like(t)
    f0 = inputs.prim_to_cons(t, vel[0] * one, vel[1] * one, vel[2] * one, one.clone(), G53)
    dh, dt = 1.0 / n, 0.3 / n
    new, r = oracle_step(oracle_mod, f0, dt, dh, G53, VL, PLM, solver)
    assert r["stats"]["n_pred_revert"] == 0 and r["stats"]["n_roe_fallback"] == 0
    ref = _vl_contact_reference(rho, vel, dt / dh)
    assert np.abs(new[0].numpy() - ref).max() <= 5e-14
    mhm, _ = oracle_step(oracle_mod, f0, dt, dh, G53, MHM, PLM, solver)
    assert (new[0] - mhm[0]).abs().max().item() > 1e-4       # and it is not the Hancock predictor


def test_vl_smooth_advection_is_second_order(oracle_mod):
    """L1 order >= 1.8 on a diagonally advected density wave (theta = 2 as in the CTU convergence pin): a predictor
    that is missing or taken over the wrong interval leaves a first-order error in time."""
    vel, t_end = (1.0, 0.75, 0.0), 0.25
    opts = oracle_mod.make_opts(theta=2.0)
    errs = []
    for n in (32, 64):
        x = ((np.arange(n) + 0.5) / n)[None, None, :]
        y = ((np.arange(n) + 0.5) / n)[None, :, None]
        rho_fn = lambda xx, yy: 1.0 + 0.3 * np.sin(2 * np.pi * (xx + yy))
        t = torch.from_numpy(np.broadcast_to(rho_fn(x, y), (16, n, n)).copy())
        one = torch.ones_like(t)
        f = inputs.prim_to_cons(t, vel[0] * one, vel[1] * one, 0.0 * one, one.clone(), 1.4)
        out, _ = oracle_run(oracle_mod, f, t_end, 1.0 / n, 1.4, 0.8, VL, PLM, HLLC, opts)
        exact = np.broadcast_to(rho_fn(x - vel[0] * t_end, y - vel[1] * t_end), (16, n, n))
        errs.append(np.abs(out[0].numpy() - exact).mean())
    assert math.log(errs[0] / errs[1], 2.0) >= 1.8, errs


def test_vl_with_ppm_is_refused(oracle_mod):
    """VL + PPM needs a fourth ghost zone; the boundary fixes three."""
    p = inputs.pack_periodic(_turb(n=16)).numpy()
    with pytest.raises(ValueError):
        oracle_mod.fluid_advance(p, 0.002, 1.0 / 16, G53, VL, PPM, HLLC)


def test_vl_cell_rebuilt_from_single_face_solves(oracle_mod):
    """General data, all five variables: the VL update of sampled cells rebuilt from oracle.riemann (pinned in
    tests/test_oracle_riemann.py) and oracle.face_values with the wiring written independently:
    first-order fluxes -> half-step state -> PLM face values of its primitives -> final fluxes -> update of U^n."""
    gamma = G53
    gm1 = gamma - 1.0
    f = _turb(n=16, seed=21)
    p = inputs.pack_periodic(f).numpy()[0]
    dh = 1.0 / 16
    dt = _dt(oracle_mod, f, dh, gamma, 0.6, VL)
    lam = dt / dh
    r = oracle_mod.fluid_advance(p[None], dt, dh, gamma, VL, PLM, HLLE)
    step = {0: (1, 0, 0), 1: (0, 1, 0), 2: (0, 0, 1)}
    sh = lambda c, d, m: tuple(c[a] + m * step[d][a] for a in range(3))
    U = lambda c: p[:, c[2], c[1], c[0]]
    memo = {}

    def f1(c, d):
        if (c, d) not in memo:
            memo[(c, d)] = oracle_mod.riemann(HLLE, d, U(c), U(sh(c, d, 1)), gamma)[0]
        return memo[(c, d)]

    def half_prim(c):
        u = U(c).copy()
        for d in range(3):
            u -= 0.5 * lam * (f1(c, d) - f1(sh(c, d, -1), d))
        v = u[1:4] / u[0]
        return np.array([u[0], v[0], v[1], v[2], gm1 * (u[4] - 0.5 * u[0] * (v ** 2).sum())])

    def face_state(c, d, side):
        strip = np.array([half_prim(sh(c, d, m)) for m in (-1, 0, 1)])
        w = np.empty(5)
        for v in range(5):
            w[v] = oracle_mod.face_values(PLM, np.array([0.0, strip[0, v], strip[1, v], strip[2, v], 0.0]))[side]
        return np.array([w[0], w[0] * w[1], w[0] * w[2], w[0] * w[3], w[4] / gm1 + 0.5 * w[0] * (w[1:4] ** 2).sum()])

    def f2(c, d):
        return oracle_mod.riemann(HLLE, d, face_state(c, d, 1), face_state(sh(c, d, 1), d, 0), gamma)[0]

    for (i, j, k) in ((0, 0, 0), (15, 7, 3), (8, 15, 12)):
        c = (i + 3, j + 3, k + 3)
        ref = U(c).copy()
        for d in range(3):
            ref -= lam * (f2(c, d) - f2(sh(c, d, -1), d))
        got = r["out"][0, :, k, j, i]
        assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max(), (i, j, k)
