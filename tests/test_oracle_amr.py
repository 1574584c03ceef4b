"""Oracle pin for the boundary fluxes: on a two-level grid, restriction plus flux correction with the
solver's `flux_out` conserve mass, momentum and energy of the composite grid to round-off; without the flux correction
they do not.  Reduced-size version of BASELINE.json config 3 (the full size runs on the GPU)."""
import torch

import amr_harness as amr

MHM, PLM, HLLE = 1, 1, 3
G53 = 5.0 / 3.0


def test_flux_correction_conserves_composite_grid(oracle_mod):
    uc, uf, region, dh_c = amr.sedov_two_level(32, 64, 64, e_blast=5.7e-5, p_amb=1.0)
    # put the (mild, P_blast ~ 10 P_ambient) blast at the coarse-fine interface so that fluxes through it are non-trivial
    uf = torch.roll(uf, shifts=(0, 0, 31), dims=(1, 2, 3))
    z0, z1, y0, y1, x0, x1 = region
    uc[:, z0:z1, y0:y1, x0:x1] = amr.restrict(uf)
    opts = oracle_mod.make_opts(min_pres=1e-10)

    def solver(p, dt, dh):
        r = oracle_mod.fluid_advance(p.numpy(), dt, dh, G53, MHM, PLM, HLLE, opts)
        return torch.from_numpy(r["out"]), torch.from_numpy(r["flux"])

    tot0 = amr.composite_total(uc, uf, region, dh_c)
    dt_c = 0.3 * dh_c / 12.0          # sound speed of the blast cells ~ 4
    for _ in range(3):
        uc, uf, rec = amr.two_level_step(solver, uc, uf, region, dh_c, dt_c)
    tot1 = amr.composite_total(uc, uf, region, dh_c)
    scale = tot0.abs() + 1e-6
    assert ((tot1 - tot0).abs() / scale).max().item() <= 1e-12
    # the interface did carry flux (otherwise the test would be vacuous)
    flux_f = rec["fine1"][2]
    assert flux_f.reshape(-1, 3, 3, 5, 16, 16)[:, 0, 2, 4].abs().max().item() > 1.0
    # and restriction alone (no flux correction) does not conserve
    uc2, uf2, region2, _ = amr.sedov_two_level(32, 64, 64, e_blast=5.7e-5, p_amb=1.0)
    uf2 = torch.roll(uf2, shifts=(0, 0, 31), dims=(1, 2, 3))
    uc2[:, z0:z1, y0:y1, x0:x1] = amr.restrict(uf2)
    t0 = amr.composite_total(uc2, uf2, region, dh_c)

    def no_flux(p, dt, dh):
        o, f = solver(p, dt, dh)
        return o, torch.zeros_like(f)

    for _ in range(3):
        uc2, uf2, _ = amr.two_level_step(no_flux, uc2, uf2, region, dh_c, dt_c)
    t1 = amr.composite_total(uc2, uf2, region, dh_c)
    assert ((t1 - t0).abs() / scale)[4].item() > 1e-9
