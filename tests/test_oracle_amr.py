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


def test_oracle_fixup_functions_in_group_layout(oracle_mod):
    """Pins oracle.restrict / oracle.flux_correct (the C loops the CUDA fix-up kernels are compared with):
    (a) restriction = the block mean (numpy reshape, an independent formulation), exact for a linear field, and it
    conserves the sum; (b) with them in place of the harness's own global-array fix-up the two-level step gives the
    same coarse level to round-off and conserves the composite grid (L112)."""
    import numpy as np
    rng = np.random.default_rng(5)
    fine = rng.standard_normal((16, 5, 16, 16, 16))
    coarse = np.zeros((2, 5, 16, 16, 16))
    parent = np.arange(16, dtype=np.int32)                       # fine group g -> octant g of coarse group g // 8
    oracle_mod.restrict(fine, coarse, parent)
    for g in range(16):
        oz, oy, ox = (g >> 2) & 1, (g >> 1) & 1, g & 1
        blk = fine[g].reshape(5, 8, 2, 8, 2, 8, 2).mean(axis=(2, 4, 6))
        got = coarse[g >> 3][:, oz * 8:oz * 8 + 8, oy * 8:oy * 8 + 8, ox * 8:ox * 8 + 8]
        assert np.abs(got - blk).max() <= 2e-15      # summation order differs from numpy.mean
    assert abs(coarse.sum() * 8 - fine.sum()) <= 1e-10
    z, y, x = np.meshgrid(np.arange(16.0), np.arange(16.0), np.arange(16.0), indexing="ij")
    lin = (1.0 + 2.0 * z - 3.0 * y + 0.5 * x)[None, None]
    c1 = np.zeros((1, 1, 16, 16, 16))
    oracle_mod.restrict(lin, c1, np.array([5], dtype=np.int32))  # octant (1, 0, 1)
    zc, yc, xc = np.meshgrid(np.arange(8.0), np.arange(8.0), np.arange(8.0), indexing="ij")
    assert np.abs(c1[0, 0, 8:, :8, 8:] - (1.0 + 2.0 * (2 * zc + 0.5) - 3.0 * (2 * yc + 0.5) + 0.5 * (2 * xc + 0.5))).max() <= 1e-13
    assert c1[0, 0, :8].max() == 0.0                              # nothing outside the octant is touched

    uc, uf, region, dh_c = amr.sedov_two_level(32, 64, 64, e_blast=5.7e-5, p_amb=1.0)
    uf = torch.roll(uf, shifts=(0, 0, 31), dims=(1, 2, 3))
    z0, z1, y0, y1, x0, x1 = region
    uc[:, z0:z1, y0:y1, x0:x1] = amr.restrict(uf)
    opts = oracle_mod.make_opts(min_pres=1e-10)

    def solver(p, dt, dh):
        r = oracle_mod.fluid_advance(p.numpy(), dt, dh, G53, MHM, PLM, HLLE, opts)
        return torch.from_numpy(r["out"]), torch.from_numpy(r["flux"])

    fix = amr.fixup_in_group_layout(
        lambda f, c, par: torch.from_numpy(oracle_mod.restrict(f.numpy(), c.numpy().copy(), par.numpy())),
        lambda acc, f, w: (w * f if acc is None else acc + w * f),
        lambda c, fc, ff, tab, lam: torch.from_numpy(oracle_mod.flux_correct(c.numpy().copy(), fc.numpy(), ff.numpy(), tab.numpy(), lam)))
    dt_c = 0.3 * dh_c / 12.0
    tot0 = amr.composite_total(uc, uf, region, dh_c)
    ua, fa, _ = amr.two_level_step(solver, uc, uf, region, dh_c, dt_c)
    ub, fb, _ = amr.two_level_step(solver, uc, uf, region, dh_c, dt_c, fixup=fix)
    assert torch.equal(fa, fb)
    assert ((ua - ub).abs().amax(dim=(1, 2, 3)) <= 1e-14 * ua.abs().amax(dim=(1, 2, 3))).all()
    assert (ua - uc).abs().max().item() > 1e-6
    tot1 = amr.composite_total(ub, fb, region, dh_c)
    assert ((tot1 - tot0).abs() / (tot0.abs() + 1e-6)).max().item() <= 1e-12
