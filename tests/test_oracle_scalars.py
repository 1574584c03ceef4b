"""Pins of the oracle's passive scalars ("an arbitrary number of chemical species, which can be renormalized
after every update to ensure that the sum of their mass fractions equals unity"; R12, R27).  CPU only."""
import math

import numpy as np
import pytest
import torch

from helpers import oracle_step
from paper_1712_07070_b200 import inputs

MHM, CTU, VL = 1, 2, 3
PLM, PPM = 1, 2
ROE, HLLC, HLLE = 1, 2, 3
G53 = 5.0 / 3.0
SCHEMES = [(MHM, PLM, ROE), (MHM, PPM, HLLC), (CTU, PPM, HLLC), (CTU, PLM, HLLE), (VL, PLM, HLLC)]


def _field(ns, n=32, seed=1712, fractions=None):
    """turbulence field + ns species s_k = X_k rho; X_k smooth positive fields that sum to 1 unless `fractions` fixes
    them as constants"""
    f = inputs.turbulence_field(n, seed, kmax=4, gamma=G53)
    rho = f[0]
    if fractions is not None:
        xs = [torch.full_like(rho, float(x)) for x in fractions]
    else:
        raw = [torch.exp(0.5 * inputs.random_field(rho.shape, seed + 31 * (k + 1), 4, "cpu")) for k in range(ns)]
        tot = sum(raw)
        xs = [r / tot for r in raw]
    return torch.cat([f, torch.stack([x * rho for x in xs])], dim=0)


def _dt(oracle, field, dh, scheme, ns):
    u = inputs.interior(inputs.pack_periodic(field)).contiguous().numpy()
    return oracle.cfl_dt(u, dh, G53, 0.4, scheme, oracle.make_opts(n_scalar=ns))[0]


@pytest.mark.parametrize("scheme,recon,solver", SCHEMES)
def test_each_species_is_conserved_and_equals_its_single_scalar_run(oracle_mod, scheme, recon, solver):
    """Without renormalisation every species obeys its own conservation law: sum over the periodic box unchanged to
    round-off (L112), and -- since a scalar never feeds back on the flow nor on another scalar -- species k of a
    4-species run carries exactly the bits of a 1-species run of that species alone.  Kills index mix-ups between
    species anywhere in reconstruction, tracing, predictor, Riemann flux and update."""
    ns = 4
    f = _field(ns)
    dh = 1.0 / 32
    dt = _dt(oracle_mod, f, dh, scheme, ns)
    new, r = oracle_step(oracle_mod, f, dt, dh, G53, scheme, recon, solver, opts=oracle_mod.make_opts(n_scalar=ns))
    assert r["stats"]["n_unphysical"] == 0
    for v in range(5 + ns):
        s0, s1 = math.fsum(f[v].flatten().tolist()), math.fsum(new[v].flatten().tolist())
        assert abs(s1 - s0) <= 1e-13 * (math.fsum(f[v].abs().flatten().tolist()) + 1.0), v
    hydro, _ = oracle_step(oracle_mod, f[:5].contiguous(), dt, dh, G53, scheme, recon, solver)
    assert torch.equal(new[:5], hydro)                       # the scalars do not touch the flow
    for k in (0, 2, 3):
        one = torch.cat([f[:5], f[5 + k:6 + k]], dim=0).contiguous()
        single, _ = oracle_step(oracle_mod, one, dt, dh, G53, scheme, recon, solver, opts=oracle_mod.make_opts(n_scalar=1))
        assert torch.equal(single[5], new[5 + k]), k
    assert (new[5:] - f[5:]).abs().max() > 1e-3


@pytest.mark.parametrize("scheme,recon,solver", SCHEMES)
def test_uniform_mass_fractions_stay_uniform(oracle_mod, scheme, recon, solver):
    """s_k = X_k rho with constant X_k: the scalar equation is X_k times the continuity equation, so s_k / rho must stay
    X_k.  Not bitwise: the predictor forms X_k rho_face - dt/2dh (X_k a - X_k b), which rounds differently from
    X_k (rho_face - dt/2dh (a - b)); a few ulp."""
    xs = (0.5, 0.3, 0.2)
    f = _field(3, fractions=xs)
    dh = 1.0 / 32
    dt = _dt(oracle_mod, f, dh, scheme, 3)
    new, _ = oracle_step(oracle_mod, f, dt, dh, G53, scheme, recon, solver, opts=oracle_mod.make_opts(n_scalar=3))
    for k, x in enumerate(xs):
        assert ((new[5 + k] / new[0] - x).abs().max().item()) <= 2e-14
    assert (new[0] - f[0]).abs().max() > 1e-3


@pytest.mark.parametrize("scheme,recon,solver", [(MHM, PLM, ROE), (CTU, PPM, HLLC), (VL, PLM, HLLC)])
def test_renormalisation_makes_the_fractions_sum_to_one(oracle_mod, scheme, recon, solver):
    """L96.  Limited reconstruction of each species on its own lets sum_k s_k drift from rho (measured ~1e-3 here);
    with `renormalize` it is rho again to round-off, each species is the unrenormalised one times rho / sum -- the
    closed form -- and the flow variables are untouched."""
    ns = 4
    f = _field(ns, seed=99)
    dh = 1.0 / 32
    dt = _dt(oracle_mod, f, dh, scheme, ns)
    raw, _ = oracle_step(oracle_mod, f, dt, dh, G53, scheme, recon, solver, opts=oracle_mod.make_opts(n_scalar=ns))
    ren, _ = oracle_step(oracle_mod, f, dt, dh, G53, scheme, recon, solver,
                         opts=oracle_mod.make_opts(n_scalar=ns, renormalize=True))
    drift = (raw[5:].sum(0) / raw[0] - 1.0).abs().max().item()
    assert drift > 1e-6                                       # there is something to renormalise
    assert (ren[5:].sum(0) / ren[0] - 1.0).abs().max().item() <= 1e-15       # 4 species: a few ulp
    assert torch.equal(ren[:5], raw[:5])
    expect = raw[5:] * (raw[0] / raw[5:].sum(0))[None]
    assert ((ren[5:] - expect).abs().max().item()) <= 1e-15 * expect.abs().max().item()


def test_renormalisation_closed_form_and_entropy_is_left_out(oracle_mod):
    """Hand values through the closing step of one cell: rho = 2, species (0.5, 0.7, 0.9) -> times 2 / 2.1.  With the
    dual-energy formalism the LAST scalar is the entropy (L100): it is not a mass fraction and keeps its value."""
    rho, v, p = 2.0, np.array([0.3, -0.2, 0.1]), 1.5
    e = p / (G53 - 1.0) + 0.5 * rho * (v ** 2).sum()
    U = np.array([rho, *(rho * v), e, 0.5, 0.7, 0.9])
    out, ok, _ = oracle_mod.close_cell(U, G53, oracle_mod.make_opts(n_scalar=3, renormalize=True))
    assert ok and np.array_equal(out[:5], U[:5])
    assert np.abs(out[5:] - np.array([0.5, 0.7, 0.9]) * (2.0 / 2.1)).max() <= 2e-16
    # without the flag nothing happens
    out, _, _ = oracle_mod.close_cell(U, G53, oracle_mod.make_opts(n_scalar=3))
    assert np.array_equal(out, U)
    # dual energy: 2 species + entropy; E_the / E_kin is large here, so the entropy is resynchronised from E (R13)
    s_ent = p / rho ** (G53 - 1.0)
    U2 = np.array([rho, *(rho * v), e, 0.8, 0.6, 123.0])
    out, ok, st = oracle_mod.close_cell(U2, G53, oracle_mod.make_opts(n_scalar=3, dual_energy=True, renormalize=True))
    assert ok and st["n_dual_fix"] == 0
    assert np.abs(out[5:7] - np.array([0.8, 0.6]) * (2.0 / 1.4)).max() <= 4e-16
    assert out[7] == pytest.approx(s_ent, rel=1e-15)
    # a non-positive sum is left alone
    U3 = np.array([rho, *(rho * v), e, 0.0, 0.0])
    out, _, _ = oracle_mod.close_cell(U3, G53, oracle_mod.make_opts(n_scalar=2, renormalize=True))
    assert np.array_equal(out, U3)


def test_scalar_count_limits(oracle_mod):
    p = inputs.pack_periodic(_field(8, n=16)).numpy()
    r = oracle_mod.fluid_advance(p, 1e-3, 1.0 / 16, G53, MHM, PLM, HLLC, oracle_mod.make_opts(n_scalar=8))
    assert np.isfinite(r["out"]).all()
    with pytest.raises(ValueError):
        oracle_mod.fluid_advance(np.zeros((1, 14, 22, 22, 22)), 1e-3, 1.0, G53, MHM, PLM, HLLC, oracle_mod.make_opts(n_scalar=9))
