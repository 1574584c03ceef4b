"""Oracle pin for the boundary fluxes: on a two-level grid, restriction plus flux correction with the
solver's `flux_out` conserve mass, momentum and energy of the composite grid to round-off; without the flux correction
they do not.  Reduced-size version of BASELINE.json config 3 (the full size runs on the GPU)."""
import pytest
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


def _two_level_random(seed=11):
    """32^3 coarse periodic level, refined region = its central 16^3 coarse cells (2x2x2 fine groups), smooth random data."""
    import numpy as np
    from paper_1712_07070_b200 import inputs
    uc = inputs.turbulence_field(32, seed, kmax=4, gamma=G53)
    uf = inputs.turbulence_field(32, seed + 1, kmax=4, gamma=G53)
    region = (8, 24, 8, 24, 8, 24)
    parent, _ = amr.region_tables(region, uc.shape[1:])
    nbr = amr.region_neighbors(region)
    return uc, uf, region, parent.numpy(), nbr.numpy()


def _oracle_pack_fine(oracle_mod, uc_pad, uf, parent, nbr, **kw):
    import numpy as np
    ug = amr.to_groups(uf).numpy()
    padded = np.full((ug.shape[0], ug.shape[1], 22, 22, 22), np.nan)
    padded[:, :, 3:19, 3:19, 3:19] = ug
    oracle_mod.fill_ghosts_table(ug, nbr, padded)
    return oracle_mod.interpolate_ghosts(uc_pad, parent, nbr, padded, **kw)


def test_interpolated_ghosts_match_the_global_array_harness(oracle_mod):
    """oracle.interpolate_ghosts (per-group index arithmetic, L248 / reading R24) against the independent whole-array
    formulation of the harness (amr.pack_fine: shifted-array central slopes on the global coarse array, strided child
    assignment): the complete padded fine batch agrees, so octant offsets, child parity, signs and axis order are right;
    every ghost cell is written (no NaN left) and sibling slabs keep the sibling copy."""
    import numpy as np
    from paper_1712_07070_b200 import inputs
    uc, uf, region, parent, nbr = _two_level_random()
    ref, _ = amr.pack_fine(uf, uc, region)
    got = _oracle_pack_fine(oracle_mod, inputs.pack_periodic(uc).numpy(), uf, parent, nbr)
    assert not np.isnan(got).any()
    assert np.abs(got - ref.numpy()).max() <= 1e-15 * np.abs(ref.numpy()).max()
    # linear in time: blending two coarse levels = interpolating from the blended level
    uc2 = inputs.turbulence_field(32, 5, kmax=4, gamma=G53)
    ref_t, _ = amr.pack_fine(uf, 0.75 * uc + 0.25 * uc2, region)
    got_t = _oracle_pack_fine(oracle_mod, inputs.pack_periodic(uc).numpy(), uf, parent, nbr,
                              coarse_padded_new=inputs.pack_periodic(uc2).numpy(), w=0.25)
    assert np.abs(got_t - ref_t.numpy()).max() <= 1e-14 * np.abs(ref_t.numpy()).max()


@pytest.mark.parametrize("monotonic", [False, True])
def test_interpolated_ghosts_linear_exactness_conservation_and_bounds(oracle_mod, monotonic):
    """What the mathematics fixes for a conservative linear interpolation: (a) data linear in (x,y,z) is reproduced
    exactly at the fine cell centres by both slope choices; (b) the two children of a coarse cell along an axis average to
    the parent, so complete 2x2x2 child sets (the two inner ghost layers of the face slabs) conserve it; (c) with
    minmod slopes no child leaves the range spanned by its parent and the parent's six face neighbours."""
    import numpy as np
    from paper_1712_07070_b200 import inputs
    uc, uf, region, parent, nbr = _two_level_random()
    # (a) linear data on one coarse group (no periodic wrap inside the stencil): value = 1 + 2x + 3y - 4z at coarse centres
    zc, yc, xc = np.meshgrid(*(np.arange(-3, 19) + 0.5,) * 3, indexing="ij")
    lin = (1 + 2 * xc + 3 * yc - 4 * zc)[None, None].repeat(5, 1)
    pad = np.full((8, 5, 22, 22, 22), np.nan)
    none = np.full((8, 27), -1, dtype=np.int32)
    oracle_mod.interpolate_ghosts(lin, np.arange(8, dtype=np.int32), none, pad, monotonic=monotonic)
    for o in range(8):
        oz, oy, ox = o >> 2, (o >> 1) & 1, o & 1
        zf, yf, xf = np.meshgrid(*(((np.arange(-3, 19) + 0.5) / 2 + 8 * q) for q in (oz, oy, ox)), indexing="ij")
        want = 1 + 2 * xf + 3 * yf - 4 * zf
        ghost = np.ones((22, 22, 22), bool)
        ghost[3:19, 3:19, 3:19] = False
        assert np.isnan(pad[o, 0][~ghost]).all()                       # interior never written
        assert np.abs(pad[o, 0][ghost] - want[ghost]).max() <= 1e-13
    # (b), (c) on random data
    cp = inputs.pack_periodic(uc).numpy()
    got = _oracle_pack_fine(oracle_mod, cp, uf, parent, nbr, monotonic=monotonic)
    for g in range(8):
        cg, o = parent[g] >> 3, parent[g] & 7
        oz, oy, ox = o >> 2, (o >> 1) & 1, o & 1
        if nbr[g, 4] < 0:                                               # low-z face slab: fine k = -2,-1 <-> coarse k = 8 oz - 1
            blk = got[g][:, 1:3, 3:19, 3:19].reshape(5, 2, 8, 2, 8, 2).mean(axis=(1, 3, 5))
            par = cp[cg][:, 8 * oz - 1 + 3, 8 * oy + 3:8 * oy + 11, 8 * ox + 3:8 * ox + 11]
            assert np.abs(blk - par).max() <= 1e-14 * np.abs(par).max()
        if nbr[g, 14] < 0:                                              # high-x face slab: fine i = 16,17 <-> coarse i = 8 ox + 8
            blk = got[g][:, 3:19, 3:19, 19:21].reshape(5, 8, 2, 8, 2, 2).mean(axis=(2, 4, 5))
            par = cp[cg][:, 8 * oz + 3:8 * oz + 11, 8 * oy + 3:8 * oy + 11, 8 * ox + 8 + 3]
            assert np.abs(blk - par).max() <= 1e-14 * np.abs(par).max()
        if monotonic and nbr[g, 12] < 0:                                # low-x face slab, every cell
            for pi in range(3):
                qi = 8 * ox + (pi - 3) // 2 + 3
                sl = (slice(None), slice(8 * oz + 3, 8 * oz + 11), slice(8 * oy + 3, 8 * oy + 11))
                C = cp[cg]
                stack = np.stack([C[:, 8 * oz + 3 + a:8 * oz + 11 + a, 8 * oy + 3 + b:8 * oy + 11 + b, qi + c]
                                  for a, b, c in ((0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1))])
                lo, hi = stack.min(0), stack.max(0)
                child = got[g][:, 3:19, 3:19, pi].reshape(5, 8, 2, 8, 2)
                tol = 1e-14 * np.abs(stack).max()
                # |child - parent| <= sum_d |s_d| / 4 <= 3/4 of the largest one-sided difference: inside [lo, hi] widened by
                # the two other axes' share; the sharp statement per axis is tested on 1-D data below
                assert (child >= (lo - 0.5 * (hi - lo))[:, :, None, :, None] - tol).all()
                assert (child <= (hi + 0.5 * (hi - lo))[:, :, None, :, None] + tol).all()
    if monotonic:
        # 1-D data along x, values worked out by hand: coarse padded cells 0..3 = 0, 1, 5, 2 and 10..13 = 4, 6, 7, 7.5
        #   cell 1: minmod(1-0, 5-1) = 1    -> its upper child (fine i = -3)      = 1 + 1/4        = 1.25
        #   cell 2: local maximum, slope 0   -> both children (fine i = -2, -1)   = 5
        #   cell 11: minmod(6-4, 7-6) = 1   -> children (fine i = 16, 17)         = 5.75, 6.25
        #   cell 12: minmod(7-6, 7.5-7) = .5 -> its lower child (fine i = 18)      = 7 - 1/8        = 6.875
        prof = np.array([0.0, 1.0, 5.0, 2.0, 2.0, 2.0, 2.0, 2.0, 2.0, 2.0, 4.0, 6.0, 7.0, 7.5] + [8.0] * 8)
        one = np.broadcast_to(prof[None, None, None, None, :], (1, 5, 22, 22, 22)).copy()
        pad = np.full((1, 5, 22, 22, 22), np.nan)
        oracle_mod.interpolate_ghosts(one, np.array([0], dtype=np.int32), none[:1], pad, monotonic=True)
        assert pad[0, 0, 5, 5, :3].tolist() == [1.25, 5.0, 5.0]
        assert pad[0, 4, 0, 21, 19:].tolist() == [5.75, 6.25, 6.875]
        # the central slope of the other mode overshoots there: cell 2 has (2-1)/2 = 0.5 -> children 4.875, 5.125
        oracle_mod.interpolate_ghosts(one, np.array([0], dtype=np.int32), none[:1], pad, monotonic=False)
        assert pad[0, 0, 5, 5, :3].tolist() == [1.0 + 0.25 * 2.5, 4.875, 5.125]
