"""GPU parity for the extended entry (scalars, dual energy, floors, remedies, other limiters) and for the
BASELINE.json configurations at their full sizes (configs 2, 4, 5)."""
import math

import numpy as np
import pytest
import torch

from helpers import rel_l1
from paper_1712_07070_b200 import binding as gb
from paper_1712_07070_b200 import inputs

pytestmark = pytest.mark.gpu
G53 = 5.0 / 3.0


@pytest.fixture(scope="module")
def dev():
    assert torch.cuda.is_available()
    gb.lib()
    return torch.device("cuda:0")


def gpu_ex(padded, dt, dh, gamma, scheme, recon, solver, **kw):
    out, flux, speed = gb.alloc_outputs(padded)
    nun = torch.zeros(1, dtype=torch.int32, device=padded.device)
    diag = torch.zeros(4, dtype=torch.int32, device=padded.device)
    o = gb.make_opts(group_speed_out=speed, n_unphysical_out=nun, diag_out=diag, **kw)
    gb.gamer_fluid_advance_ex(padded, out, flux, dt, dh, gamma, scheme, recon, solver, o)
    torch.cuda.synchronize()
    return out, flux, speed, int(nun.item()), diag.cpu().tolist()


def oracle_opts(oracle, **kw):
    return oracle.make_opts(**kw)


STRESS = [
    (gb.CTU, gb.PPM, gb.HLLC, dict(n_scalar=1, dual_energy=True, remedy_first_order=True, min_pres=1e-12, min_dens=1e-10)),
    (gb.CTU, gb.PPM, gb.ROE, dict(n_scalar=1, dual_energy=True, remedy_first_order=True)),
    (gb.MHM, gb.PPM, gb.ROE, dict(remedy_first_order=True)),
    (gb.MHM, gb.PLM, gb.HLLE, dict(n_scalar=1, min_temp=1e-3)),
    (gb.CTU, gb.PLM, gb.ROE, dict()),
    (gb.VL, gb.PLM, gb.ROE, dict(n_scalar=1, dual_energy=True, remedy_first_order=True, min_pres=1e-12, min_dens=1e-10)),
    (gb.VL, gb.PLM, gb.HLLC, dict()),
]


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("scheme,recon,solver,kw", STRESS)
def test_stress_modes_match_oracle(dev, oracle_mod, scheme, recon, solver, kw, dtype):
    """Mach-10, sigma=2 turbulence: every discontinuous decision (remedy (i), reverts, remedy (ii), dual-energy
    switch) is exercised; fp64 must take the same decisions as the oracle, fp32 may differ on marginal ones."""
    ent = kw.get("n_scalar", 0) == 1
    f = inputs.turbulence_field(32, 3, kmax=6, gamma=G53, mach=10.0, sigma=2.0, entropy=ent)
    padded = inputs.pack_periodic(f).to(dtype)
    p64 = padded.to(torch.float64)
    dh = 1 / 32
    dt = oracle_mod.cfl_dt(inputs.interior(p64).contiguous().numpy(), dh, G53, 0.45, scheme,
                           oracle_mod.make_opts(n_scalar=int(ent)))[0]
    ref = oracle_mod.fluid_advance(p64.numpy(), dt, dh, G53, scheme, recon, solver, oracle_mod.make_opts(**kw))
    out, flux, speed, nun, diag = gpu_ex(padded.to(dev), dt, dh, G53, scheme, recon, solver, **kw)
    st = ref["stats"]
    err = rel_l1(out.cpu().numpy(), ref["out"], G53)
    if dtype == torch.float64:
        assert nun == st["n_unphysical"]
        # per-cell decisions are counted exactly; per-face / per-state ones are counted once per tile, and the
        # fp64 variants that do not fit 227 KB split a group in 2 or 4 tiles whose halo faces overlap
        assert diag[2] == st["n_first_order"] and diag[3] == st["n_dual_fix"]
        # (VL: the half-step predictor of a 4-row tile covers 8 rows, so its first-pass faces are counted twice)
        over = 2.2 if scheme == gb.VL else 1.6
        assert st["n_roe_fallback"] <= diag[0] <= over * st["n_roe_fallback"] + 2
        assert 0.9 * st["n_pred_revert"] - 2 <= diag[1] <= over * st["n_pred_revert"] + 2
        assert max(err.values()) <= 1e-12, err
        fe = np.abs(flux.cpu().numpy() - ref["flux"]).sum() / np.abs(ref["flux"]).sum()
        assert fe <= 1e-12
        assert np.abs(speed.cpu().numpy() - ref["speed"]).max() <= 1e-11 * ref["speed"].max()
    else:
        # fp32: the continuous arithmetic must meet the contract's 1e-5; what may differ from the fp64 oracle are the
        # DISCONTINUOUS decisions on marginal data (remedy (i) fallback, predictor / correction reverts, remedy (ii), the
        # dual-energy switch): SURVEY 8(c) asks for their number.  A cell counts as "decided differently" when it is off by
        # more than 1e-3 of the variable's scale (three orders above fp32 round-off, the size of a flipped decision);
        # the 1e-5 bound is asserted on all other cells, the differing cells are counted, bounded and reported.
        o, r = out.cpu().numpy().astype(np.float64), ref["out"]
        scale = np.abs(r).mean(axis=(0, 2, 3, 4), keepdims=True) + 1e-300
        scale[:, 1:4] = np.sqrt((r[:, 1:4] ** 2).sum(axis=1, keepdims=True)).mean() + np.abs(r[:, 0:1]).mean() * math.sqrt(G53)
        cell_err = (np.abs(o - r) / scale).max(axis=1)                   # [G,16,16,16]
        differ = cell_err > 1e-3
        n_diff, n_cells = int(differ.sum()), differ.size
        keep = ~differ
        agree = {name: np.abs(o[:, v][keep] - r[:, v][keep]).sum() / np.abs(r[:, v][keep]).sum() for v, name in ((0, "rho"), (4, "E"))}
        agree["mom"] = sum(np.abs(o[:, d][keep] - r[:, d][keep]).sum() for d in (1, 2, 3)) / (scale[0, 1, 0, 0, 0] * keep.sum())
        counts = {"cells_decided_differently": n_diff, "of": n_cells,
                  "remedy_i_faces": (diag[0], st["n_roe_fallback"]), "reverted_states": (diag[1], st["n_pred_revert"]),
                  "remedy_ii_cells": (diag[2], st["n_first_order"]), "dual_energy_cells": (diag[3], st["n_dual_fix"]),
                  "unphysical": (nun, st["n_unphysical"])}
        print("fp32 decisions (gpu, oracle):", counts, "L1 on agreeing cells:", agree)
        assert max(agree.values()) <= 1e-5, (agree, counts)
        assert n_diff <= 2e-3 * n_cells, counts                          # measured: a few 1e-4 of the cells at Mach 10
        assert abs(nun - st["n_unphysical"]) <= 2 + 0.02 * st["n_unphysical"], counts
        assert abs(diag[2] - st["n_first_order"]) <= 3 + 0.05 * st["n_first_order"], counts
        assert abs(diag[3] - st["n_dual_fix"]) <= 3 + 0.02 * st["n_dual_fix"], counts
        assert max(err.values()) <= 2e-4, err                            # and the flipped cells stay far below O(1) in the norm
    assert torch.isfinite(out).all()


@pytest.mark.parametrize("limiter", [gb.VANLEER, gb.VANALBADA])
@pytest.mark.parametrize("recon", [gb.PLM, gb.PPM])
def test_other_limiters(dev, oracle_mod, limiter, recon):
    f = inputs.turbulence_field(32, 9, kmax=4, gamma=G53)
    padded = inputs.pack_periodic(f)
    dh, dt = 1 / 32, 0.003
    ref = oracle_mod.fluid_advance(padded.numpy(), dt, dh, G53, gb.MHM, recon, gb.HLLC, oracle_mod.make_opts(limiter=limiter))
    out = gpu_ex(padded.to(dev), dt, dh, G53, gb.MHM, recon, gb.HLLC, limiter=limiter)[0]
    assert max(rel_l1(out.cpu().numpy(), ref["out"], G53).values()) <= 1e-12
    base = gpu_ex(padded.to(dev), dt, dh, G53, gb.MHM, recon, gb.HLLC)[0]
    assert not torch.equal(base, out)


def test_config5_stress_disk_fp64_dual_energy(dev, oracle_mod):
    """BASELINE.json config 5 at reduced extent (64 x 64 x 32 cells = 32 groups; the full 8192-group batch is
    sampled in test_config5_full_size_sampled)."""
    f = inputs.disk_field(64, 64, 32, 2018, gamma=G53)
    padded = inputs.pack_periodic(f)
    kw = dict(n_scalar=1, dual_energy=True, de_xi=1e-2, min_temp=1e-3, min_dens=1e-8, remedy_first_order=True)
    dh = 1 / 64
    dt = oracle_mod.cfl_dt(inputs.interior(padded).contiguous().numpy(), dh, G53, 0.4, gb.CTU, oracle_mod.make_opts(n_scalar=1))[0]
    ref = oracle_mod.fluid_advance(padded.numpy(), dt, dh, G53, gb.CTU, gb.PPM, gb.HLLC, oracle_mod.make_opts(**kw))
    out, flux, speed, nun, diag = gpu_ex(padded.to(dev), dt, dh, G53, gb.CTU, gb.PPM, gb.HLLC, **kw)
    o = out.cpu().numpy()
    assert np.isfinite(o).all() and (o[:, 0] > 0).all()
    pres = (G53 - 1) * (o[:, 4] - 0.5 * (o[:, 1] ** 2 + o[:, 2] ** 2 + o[:, 3] ** 2) / o[:, 0])
    assert (pres > 0).all() and nun == ref["stats"]["n_unphysical"] == 0
    assert max(rel_l1(o, ref["out"], G53).values()) <= 1e-12
    assert diag[3] == ref["stats"]["n_dual_fix"] and diag[3] > 1000
    assert diag[2] == ref["stats"]["n_first_order"]


def _sampled_parity(dev, oracle_mod, field, dtype, scheme, recon, solver, cfl, tol, kw=None, n_sample=48):
    """Full-size batch in the launch configuration bench.py times; oracle on sampled groups (first, last, spread)."""
    kw = kw or {}
    padded = inputs.pack_periodic(field, dtype=dtype)
    g = padded.shape[0]
    n = field.shape[-1]
    dh = 1.0 / n
    dt_dev = torch.zeros(1, dtype=torch.float64, device=dev)
    gb.gamer_cfl_dt(inputs.interior(padded).contiguous(), dh, G53, cfl, scheme, None, dt_dev,
                    gb.make_opts(n_scalar=kw.get("n_scalar", 0)))
    dt = float(dt_dev.item())
    out, flux, speed, nun, diag = gpu_ex(padded, dt, dh, G53, scheme, recon, solver, **kw)
    idx = np.unique(np.concatenate([[0, 1, g - 1], np.linspace(0, g - 1, n_sample).astype(np.int64)]))
    sel = torch.from_numpy(idx).to(dev)
    samp = padded[sel].to(torch.float64).cpu().numpy()
    ref = oracle_mod.fluid_advance(samp, dt, dh, G53, scheme, recon, solver, oracle_mod.make_opts(**kw))
    err = rel_l1(out[sel].cpu().numpy(), ref["out"], G53)
    assert max(err.values()) <= tol, err
    fe = np.abs(flux[sel].cpu().numpy() - ref["flux"]).sum() / np.abs(ref["flux"]).sum()
    assert fe <= 2 * tol
    assert np.abs(speed[sel].cpu().numpy() - ref["speed"]).max() <= max(tol, 2e-6 if dtype == torch.float32 else 0) * ref["speed"].max()
    # the dt the GPU computed is the CFL formula evaluated on the whole batch
    assert torch.isfinite(out).all()
    # property that holds at any size: conservation on the periodic box (fp64 accumulation of the outputs)
    tot0 = inputs.interior(padded).to(torch.float64).sum(dim=(0, 2, 3, 4))
    tot1 = out.to(torch.float64).sum(dim=(0, 2, 3, 4))
    scale = inputs.interior(padded).to(torch.float64).abs().sum(dim=(0, 2, 3, 4))
    rel = ((tot1 - tot0).abs() / scale)[:5].max().item()
    assert rel <= (1e-13 if dtype == torch.float64 else 2e-7), rel
    return out, padded, dt


def test_config2_smooth_random_4096_groups_ctu_ppm_hllc_fp32(dev, oracle_mod):
    """BASELINE.json config 2 at full size: 256^3, CTU+PPM+HLLC fp32, one step; conservation and sampled parity;
    the whole batch is also compared (the oracle finishes 4096 groups in seconds)."""
    f = inputs.turbulence_field(256, 1712, kmax=8, gamma=G53, device=dev)
    out, padded, dt = _sampled_parity(dev, oracle_mod, f, torch.float32, gb.CTU, gb.PPM, gb.HLLC, 0.5, 1e-5)
    ref = oracle_mod.fluid_advance(padded.to(torch.float64).cpu().numpy(), dt, 1 / 256, G53, gb.CTU, gb.PPM, gb.HLLC,
                                   want_flux=False)
    assert max(rel_l1(out.cpu().numpy(), ref["out"], G53).values()) <= 1e-5


@pytest.mark.parametrize("scheme,recon,solver,cfl", [(gb.MHM, gb.PLM, gb.ROE, 0.5), (gb.CTU, gb.PPM, gb.HLLC, 0.4)])
def test_config4_full_size_sampled_fp32(dev, oracle_mod, scheme, recon, solver, cfl):
    """BASELINE.json config 4: 32,768 groups (512^3), the batch bench.py times."""
    f = inputs.turbulence_field(512, 7070, kmax=16, gamma=G53, device=dev)
    _sampled_parity(dev, oracle_mod, f, torch.float32, scheme, recon, solver, cfl, 1e-5)


@pytest.mark.parametrize("scheme,recon,solver,cfl", [(gb.MHM, gb.PLM, gb.ROE, 0.5), (gb.CTU, gb.PPM, gb.HLLC, 0.4)])
def test_config4_full_size_sampled_fp64(dev, oracle_mod, scheme, recon, solver, cfl):
    """BASELINE.json config 4 in fp64 at its full 32,768 groups (in + out + flux_out = 22 GB of the 180), both variants the
    bench times; oracle on sampled groups, conservation over the whole box."""
    f = inputs.turbulence_field(512, 7070, kmax=16, gamma=G53, device=dev)
    _sampled_parity(dev, oracle_mod, f, torch.float64, scheme, recon, solver, cfl, 1e-12, n_sample=24)


def test_config5_full_size_sampled(dev, oracle_mod):
    """BASELINE.json config 5 at full size: 512 x 512 x 128 cells = 8192 groups, fp64, dual energy."""
    f = inputs.disk_field(512, 512, 128, 2018, gamma=G53, device=dev)
    kw = dict(n_scalar=1, dual_energy=True, de_xi=1e-2, min_temp=1e-3, min_dens=1e-8, remedy_first_order=True)
    padded = inputs.pack_periodic(f)
    g, dh = padded.shape[0], 1 / 512
    assert g == 8192
    dt_dev = torch.zeros(1, dtype=torch.float64, device=dev)
    gb.gamer_cfl_dt(inputs.interior(padded).contiguous(), dh, G53, 0.4, gb.CTU, None, dt_dev, gb.make_opts(n_scalar=1))
    dt = float(dt_dev.item())
    out, flux, speed, nun, diag = gpu_ex(padded, dt, dh, G53, gb.CTU, gb.PPM, gb.HLLC, **kw)
    idx = np.unique(np.linspace(0, g - 1, 40).astype(np.int64))
    sel = torch.from_numpy(idx).to(dev)
    ref = oracle_mod.fluid_advance(padded[sel].cpu().numpy(), dt, dh, G53, gb.CTU, gb.PPM, gb.HLLC, oracle_mod.make_opts(**kw))
    assert max(rel_l1(out[sel].cpu().numpy(), ref["out"], G53).values()) <= 1e-12
    assert torch.isfinite(out).all() and (out[:, 0] > 0).all() and nun == 0
    ek = 0.5 * (out[:, 1] ** 2 + out[:, 2] ** 2 + out[:, 3] ** 2) / out[:, 0]
    assert ((out[:, 4] - ek) > 0).all()


def test_config3_two_level_sedov_flux_correction(dev, oracle_mod):
    """BASELINE.json config 3 at full size: coarse 256 x 256 x 128 cells (2048 groups) + the central half refined
    by 2 (2048 fine groups), Sedov blast (E = 1 in the central 2x2x2 fine cells, ambient rho = 1, P = 1e-5),
    MHM+PLM+HLLE through the extended entry with a tiny pressure floor; one coarse step and two fine steps, every
    batch compared with the oracle, and the composite grid conserved to round-off after restriction + flux
    correction with the GPU's flux_out."""
    import amr_harness as amr
    uc, uf, region, dh_c = amr.sedov_two_level(128, 256, 256, gamma=G53, device=dev)
    kw = dict(min_pres=1e-10)

    def gpu_solver(p, dt, dh):
        out, flux, speed, nun, diag = gpu_ex(p.contiguous(), dt, dh, G53, gb.MHM, gb.PLM, gb.HLLE, **kw)
        assert nun == 0
        return out, flux

    tot0 = amr.composite_total(uc, uf, region, dh_c)
    # blast cells: P = (gamma-1) E / (8 dv) with dv = (dh_c/2)^3; the fine level sets the step (Eq. 2, C = 0.4)
    pb = (G53 - 1.0) / (8 * (0.5 * dh_c) ** 3)
    dt_c = 2 * 0.4 * (0.5 * dh_c) / (3.0 * math.sqrt(G53 * pb))
    uc1, uf1, rec = amr.two_level_step(gpu_solver, uc, uf, region, dh_c, dt_c)
    tot1 = amr.composite_total(uc1, uf1, region, dh_c)
    assert ((tot1 - tot0).abs() / (tot0.abs() + 1e-9)).max().item() <= 1e-12
    assert torch.isfinite(uc1).all() and torch.isfinite(uf1).all()
    n_groups = 0
    for name, (p, out, flux) in rec.items():
        dt, dh = (dt_c, dh_c) if name == "coarse" else (0.5 * dt_c, 0.5 * dh_c)
        n_groups += p.shape[0]
        ref = oracle_mod.fluid_advance(p.cpu().numpy(), dt, dh, G53, gb.MHM, gb.PLM, gb.HLLE, oracle_mod.make_opts(**kw))
        err = rel_l1(out.cpu().numpy(), ref["out"], G53)
        assert max(err.values()) <= 1e-12, (name, err)
        fe = np.abs(flux.cpu().numpy() - ref["flux"]).sum() / np.abs(ref["flux"]).sum()
        assert fe <= 1e-12, (name, fe)
    assert n_groups == 2048 + 2 * 2048
    # the blast did move energy inside the fine level
    assert (uf1[4] - uf[4]).abs().max().item() > 1.0


@pytest.mark.parametrize("dtype", [torch.float32, torch.float64])
@pytest.mark.parametrize("scheme,recon,solver,kw", [(gb.MHM, gb.PLM, gb.ROE, {}), (gb.MHM, gb.PPM, gb.HLLC, {}),
                                                    (gb.MHM, gb.PLM, gb.HLLE, dict(n_scalar=1, dual_energy=True, min_pres=1e-12)),
                                                    (gb.CTU, gb.PPM, gb.HLLC, {}), (gb.CTU, gb.PLM, gb.ROE, {}),
                                                    (gb.CTU, gb.PPM, gb.HLLE, dict(n_scalar=1, dual_energy=True, min_pres=1e-12)),
                                                    (gb.VL, gb.PLM, gb.HLLC, {}), (gb.VL, gb.PLM, gb.ROE, dict(n_scalar=1, dual_energy=True, min_pres=1e-12)),
                                                    (gb.CTU, gb.PPM, gb.HLLC, dict(n_scalar=3, renormalize=True)),
                                                    (gb.MHM, gb.PPM, gb.ROE, dict(n_scalar=2))])
def test_fused_ghost_refresh_entry_matches_the_padded_path(dev, scheme, recon, solver, kw, dtype):
    """SURVEY 8(f) NEXT-1, second half: gamer_fluid_advance_resident gathers the ghost zones from the neighbours'
    unpadded state inside the solver.  On a periodic 2 x 3 x 4 box of groups (so that -1 and +1 neighbours coincide
    along z and differ along x) it must reproduce host packing + gamer_fluid_advance_ex for out, flux_out and the
    group speeds.  The two kernels are separate template instantiations (possibly of different tile height) whose
    multiply-adds the compiler may fuse differently, so the bound is a few ulp -- 1e-6 (fp32) / 1e-13 (fp64) of each
    variable's scale, ten times below the parity bounds against the oracle; most variants agree bit for bit -- and
    the neighbour table must be the periodic one."""
    gz, gy, gx = 2, 3, 4
    f = inputs.turbulence_field(16, 4242, kmax=4, gamma=G53, shape=(gz * 16, gy * 16, gx * 16), entropy=bool(kw.get("n_scalar")))
    if kw.get("n_scalar", 0) > 1:      # species: smooth positive partial densities
        extra = [f[0] * (0.2 + 0.1 * k + 0.05 * torch.sin(6.283185307179586 * (k + 1) * torch.arange(f.shape[-1], dtype=torch.float64) / f.shape[-1]))
                 for k in range(kw["n_scalar"])]
        f = torch.cat([f[:5], torch.stack([e.expand_as(f[0]).contiguous() for e in extra])], dim=0)
    padded = inputs.pack_periodic(f).to(dtype).to(dev)
    u = inputs.interior(padded).contiguous()
    dt, dh = 0.004, 1.0 / 64
    out0, flux0, speed0 = gb.alloc_outputs(padded)
    gb.gamer_fluid_advance_ex(padded, out0, flux0, dt, dh, G53, scheme, recon, solver, gb.make_opts(group_speed_out=speed0, **kw))
    nbr = gb.gamer_neighbors_periodic(gz, gy, gx, dev)
    ref = torch.empty_like(nbr)
    for g in range(gz * gy * gx):
        bz, by, bx = g // (gy * gx), (g // gx) % gy, g % gx
        for k in range(27):
            dz, dy, dx = k // 9 - 1, (k // 3) % 3 - 1, k % 3 - 1
            ref[g, k] = (((bz + dz) % gz) * gy + (by + dy) % gy) * gx + (bx + dx) % gx
    assert torch.equal(nbr.cpu(), ref.cpu())
    out1, flux1, speed1 = gb.alloc_outputs(padded)
    gb.gamer_fluid_advance_resident(u, nbr, out1, flux1, dt, dh, G53, scheme, recon, solver, gb.make_opts(group_speed_out=speed1, **kw))
    torch.cuda.synchronize()
    assert torch.isfinite(out1).all()
    tol = 1e-13 if dtype == torch.float64 else 1e-6
    for a1, a0 in ((out1, out0), (flux1, flux0), (speed1, speed0)):
        for v in range(a0.shape[1] if a0.dim() == 5 else 1):
            x1, x0 = (a1[:, v], a0[:, v]) if a0.dim() == 5 else (a1, a0)
            assert ((x1 - x0).abs().max() <= tol * x0.abs().max()).item()
    # shared faces of neighbouring groups still carry identical bits inside the fused kernel
    fl = flux1.reshape(gz, gy, gx, 3, 3, -1, 16, 16)
    for bz, by, bx in [(0, 0, 0), (1, 2, 3), (0, 1, 2)]:
        assert torch.equal(fl[bz, by, bx, 0, 2], fl[bz, by, (bx + 1) % gx, 0, 0])
        assert torch.equal(fl[bz, by, bx, 1, 2], fl[bz, (by + 1) % gy, bx, 1, 0])
        assert torch.equal(fl[bz, by, bx, 2, 2], fl[(bz + 1) % gz, by, bx, 2, 0])


def _gpu_fixup():
    """two_level_step(fixup=...) adapter that runs restriction, flux averaging and flux correction in the library."""
    import amr_harness as amr

    def restrict_fn(fine, coarse, parent):
        coarse = coarse.clone()
        gb.gamer_restrict(fine, coarse, parent)
        return coarse

    def accumulate_fn(acc, flux, w):
        init = acc is None
        acc = torch.empty_like(flux) if init else acc
        gb.gamer_flux_accumulate(acc, flux.contiguous(), w, init)
        return acc

    def correct_fn(coarse, coarse_flux, fine_avg, table, lam):
        gb.gamer_flux_correct(coarse, coarse_flux.contiguous(), fine_avg, table, lam)
        return coarse

    return amr.fixup_in_group_layout(restrict_fn, accumulate_fn, correct_fn)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_fixup_kernels_match_oracle(dev, oracle_mod, dtype):
    """gamer_restrict / gamer_flux_accumulate / gamer_flux_correct against the
    oracle's C loops on random data, with the tables of a box-shaped refined region that touches the periodic wrap
    (so corrected cells and coarse fluxes come from other groups than the parents).  fp64: the same operations in
    the same order -> identical bits; fp32: 1e-6 of the scale."""
    import amr_harness as amr
    region = (0, 16, 8, 24, 24, 48)                  # coarse cells; z starts at the periodic boundary
    cshape = (32, 32, 48)
    parent, table = amr.region_tables(region, cshape)
    n_c, n_f = (32 // 16) * (32 // 16) * (48 // 16), parent.shape[0]
    assert n_f == 2 * 2 * 3 and table.shape[0] == 2 * (2 * 2 + 2 * 3 + 2 * 3)
    g = torch.Generator().manual_seed(11)
    fine = torch.randn((n_f, 5, 16, 16, 16), generator=g, dtype=torch.float64).to(dtype)
    coarse = torch.randn((n_c, 5, 16, 16, 16), generator=g, dtype=torch.float64).to(dtype)
    cflux = torch.randn((n_c, 3, 3, 5, 16, 16), generator=g, dtype=torch.float64).to(dtype)
    ff = [torch.randn((n_f, 3, 3, 5, 16, 16), generator=g, dtype=torch.float64).to(dtype) for _ in range(2)]
    lam = 0.37
    ref = oracle_mod.restrict(fine.double().numpy(), coarse.double().numpy().copy(), parent.numpy())
    favg = 0.5 * ff[0].double().numpy() + 0.5 * ff[1].double().numpy()
    ref = oracle_mod.flux_correct(ref, cflux.double().numpy(), favg, table.numpy(), lam)
    c_gpu = coarse.to(dev).clone()
    gb.gamer_restrict(fine.to(dev), c_gpu, parent.to(dev))
    acc = torch.empty_like(ff[0], device=dev)
    gb.gamer_flux_accumulate(acc, ff[0].to(dev), 0.5, True)
    gb.gamer_flux_accumulate(acc, ff[1].to(dev), 0.5, False)
    gb.gamer_flux_correct(c_gpu, cflux.to(dev), acc, table.to(dev), lam)
    torch.cuda.synchronize()
    got = c_gpu.cpu().double().numpy()
    assert np.abs(ref - coarse.double().numpy()).max() > 0.1          # the fix-up did change cells
    if dtype == torch.float64:
        assert np.array_equal(got, ref)
        assert np.array_equal(acc.cpu().numpy(), favg)
    else:
        assert np.abs(got - ref).max() <= 1e-6 * np.abs(ref).max()
    # cells outside the refined octants and the corrected layers are untouched
    untouched = (ref == coarse.double().numpy())
    assert np.array_equal(got[untouched], coarse.double().numpy()[untouched])


def test_config3_with_gpu_fixup(dev):
    """Config 3 (reduced to 64 x 128 x 128 coarse cells) with the whole L112 fix-up on the GPU: same coarse level as
    the harness's global-array fix-up to round-off, composite grid conserved to 1e-12."""
    import amr_harness as amr
    uc, uf, region, dh_c = amr.sedov_two_level(64, 128, 128, gamma=G53, device=dev)
    kw = dict(min_pres=1e-10)

    def gpu_solver(p, dt, dh):
        out, flux, speed, nun, diag = gpu_ex(p.contiguous(), dt, dh, G53, gb.MHM, gb.PLM, gb.HLLE, **kw)
        return out, flux

    pb = (G53 - 1.0) / (8 * (0.5 * dh_c) ** 3)
    dt_c = 2 * 0.4 * (0.5 * dh_c) / (3.0 * math.sqrt(G53 * pb))
    tot0 = amr.composite_total(uc, uf, region, dh_c)
    ua, fa, _ = amr.two_level_step(gpu_solver, uc, uf, region, dh_c, dt_c)
    ub, fb, _ = amr.two_level_step(gpu_solver, uc, uf, region, dh_c, dt_c, fixup=_gpu_fixup())
    torch.cuda.synchronize()
    assert torch.equal(fa, fb)
    assert ((ua - ub).abs().amax(dim=(1, 2, 3)) <= 1e-13 * (ua.abs().amax(dim=(1, 2, 3)) + 1e-30)).all()
    tot1 = amr.composite_total(ub, fb, region, dh_c)
    assert ((tot1 - tot0).abs() / (tot0.abs() + 1e-6)).max().item() <= 1e-12      # total momentum is 0: absolute bound there


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("scheme,recon,solver,kw", [(gb.MHM, gb.PLM, gb.ROE, {}), (gb.MHM, gb.PPM, gb.HLLC, {}),
                                                    (gb.CTU, gb.PPM, gb.HLLC, {}), (gb.CTU, gb.PLM, gb.HLLE, dict(n_scalar=1)),
                                                    (gb.MHM, gb.PLM, gb.HLLC, dict(limiter=gb.VANLEER))])
def test_characteristic_variable_limiting(dev, oracle_mod, scheme, recon, solver, kw, dtype):
    """PAPER.md L94 "applied to either primitive or characteristic variables" (DESIGN R22): slopes limited in the
    characteristic variables of each cell, against the oracle, on Mach-3 turbulence rough enough for the two ways of
    limiting to differ (after three steps that build pressure waves); the usual one-step bounds (1e-12 / 1e-5)."""
    f = inputs.turbulence_field(32, 21, kmax=8, gamma=G53, mach=3.0, sigma=1.5, entropy=bool(kw.get("n_scalar")))
    dh = 1 / 32
    # the seeded field has uniform pressure, for which every characteristic amplitude is a single primitive difference and
    # the two ways of limiting coincide: let three steps build pressure waves and shocks first
    p0 = inputs.pack_periodic(f).to(dev)
    for _ in range(3):
        dt0 = oracle_mod.cfl_dt(inputs.interior(p0).contiguous().cpu().numpy(), dh, G53, 0.3, scheme,
                                oracle_mod.make_opts(n_scalar=kw.get("n_scalar", 0)))[0]
        o0 = gpu_ex(p0, dt0, dh, G53, gb.MHM, gb.PLM, gb.HLLE, n_scalar=kw.get("n_scalar", 0))[0]
        gb.gamer_refresh_ghosts_periodic(o0, p0, 2, 2, 2)
    torch.cuda.synchronize()
    padded = p0.cpu().to(dtype)
    dt = oracle_mod.cfl_dt(inputs.interior(padded.double()).contiguous().numpy(), dh, G53, 0.3, scheme,
                           oracle_mod.make_opts(n_scalar=kw.get("n_scalar", 0)))[0]
    ref = oracle_mod.fluid_advance(padded.double().numpy(), dt, dh, G53, scheme, recon, solver,
                                   oracle_mod.make_opts(char_limiting=True, **kw))
    out, flux, speed, nun, diag = gpu_ex(padded.to(dev), dt, dh, G53, scheme, recon, solver, char_limiting=True, **kw)
    tol = 1e-12 if dtype == torch.float64 else 1e-5
    err = rel_l1(out.cpu().double().numpy(), ref["out"], G53)
    assert max(err.values()) <= tol, err
    fe = np.abs(flux.cpu().double().numpy() - ref["flux"]).sum() / np.abs(ref["flux"]).sum()
    assert fe <= 2 * tol
    base = gpu_ex(padded.to(dev), dt, dh, G53, scheme, recon, solver, **kw)[0]
    assert (base - out).abs().max().item() > 1e-3          # and it is not the primitive-variable result


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_remedy_iv_v_retry_matches_oracle(dev, oracle_mod, dtype):
    """gamer_fluid_advance_retry (remedies (iv), (v), L107-108) against oracle.fluid_advance_retry: Mach-3 turbulence with
    5x the Eq. (2) step on 8 groups; the same number of reductions, the same accepted dt (bitwise: repeated
    multiplication by 0.8 in double on both sides), the accepted result within the one-step tolerance; and the abort."""
    f = inputs.turbulence_field(32, 3, kmax=6, gamma=G53, mach=3.0, sigma=1.0)
    padded = inputs.pack_periodic(f).to(dtype)
    p64 = padded.to(torch.float64)
    dh = 1 / 32
    dt0 = 5.0 * oracle_mod.cfl_dt(inputs.interior(p64).contiguous().numpy(), dh, G53, 0.5, gb.MHM)[0]
    ref = oracle_mod.fluid_advance_retry(p64.numpy(), dt0, dh, G53, gb.MHM, gb.PLM, gb.ROE)
    assert ref["n_retries"] >= 2
    pd = padded.to(dev)
    out, flux, speed = gb.alloc_outputs(pd)
    nun = torch.zeros(1, dtype=torch.int32, device=dev)
    o = gb.make_opts(group_speed_out=speed, n_unphysical_out=nun)
    before = gb.gamer_launch_count()
    dt_used, k = gb.gamer_fluid_advance_retry(pd, out, flux, dt0, dh, G53, gb.MHM, gb.PLM, gb.ROE, o)
    assert gb.gamer_launch_count() - before >= k + 1            # every attempt is a kernel launch
    assert int(nun.item()) == 0 and torch.isfinite(out).all()
    assert k == ref["n_retries"] and dt_used == ref["dt_used"]
    err = rel_l1(out.cpu().numpy(), ref["out"], G53)
    assert max(err.values()) <= (1e-12 if dtype == torch.float64 else 1e-5), err
    fe = np.abs(flux.cpu().numpy() - ref["flux"]).sum() / np.abs(ref["flux"]).sum()
    assert fe <= (1e-12 if dtype == torch.float64 else 1e-5)
    # remedy (v): threshold above the accepted step -> GAMER_EUNPHYSICAL, as the oracle's abort
    with pytest.raises(FloatingPointError):
        oracle_mod.fluid_advance_retry(p64.numpy(), dt0, dh, G53, gb.MHM, gb.PLM, gb.ROE, dt_min=1.01 * dt_used)
    with pytest.raises(gb.GamerError, match="-4"):
        gb.gamer_fluid_advance_retry(pd, out, flux, dt0, dh, G53, gb.MHM, gb.PLM, gb.ROE, o, dt_min=1.01 * dt_used)
    assert int(nun.item()) > 0


@pytest.mark.parametrize("monotonic", [False, True])
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_interpolated_ghosts_match_oracle(dev, oracle_mod, dtype, monotonic):
    """gamer_interpolate_ghosts (L248 "interpolating from coarse patches", L482 temporal interpolation; R24) against
    oracle.interpolate_ghosts: a refined box that touches the periodic wrap of a 32 x 32 x 48 coarse level (parents in several
    coarse groups, all 8 octants), 6 variables, two coarse states blended at w = 0.25; after gamer_refresh_ghosts_table has
    copied the sibling slabs.  fp64: identical bits; fp32: 1e-6 of the scale.  Slabs with a sibling and the interior keep
    their values; a second call without the time blend is checked too."""
    import amr_harness as amr
    region = (0, 16, 8, 24, 24, 48)
    cshape = (32, 32, 48)
    parent, _ = amr.region_tables(region, cshape)
    nbr = amr.region_neighbors(region)
    n_f = parent.shape[0]
    assert n_f == 2 * 2 * 3 and sorted(set((parent % 8).tolist())) == list(range(8))
    g = torch.Generator().manual_seed(5)
    uc0 = torch.randn((6, *cshape), generator=g, dtype=torch.float64)
    uc1 = uc0 + 0.3 * torch.randn((6, *cshape), generator=g, dtype=torch.float64)
    c0, c1 = inputs.pack_periodic(uc0).to(dtype), inputs.pack_periodic(uc1).to(dtype)
    uf = torch.randn((n_f, 6, 16, 16, 16), generator=g, dtype=torch.float64).to(dtype)
    for blend in (True, False):
        ref = np.full((n_f, 6, 22, 22, 22), -7.0)
        ref[:, :, 3:19, 3:19, 3:19] = uf.double().numpy()
        oracle_mod.fill_ghosts_table(uf.double().numpy(), nbr.numpy(), ref)
        sibling_only = ref.copy()
        oracle_mod.interpolate_ghosts(c0.double().numpy(), parent.numpy(), nbr.numpy(), ref,
                                      coarse_padded_new=c1.double().numpy() if blend else None, w=0.25, monotonic=monotonic)
        assert (ref != -7.0).all() and (sibling_only == -7.0).any()
        fine = torch.full((n_f, 6, 22, 22, 22), -7.0, dtype=dtype, device=dev)
        fine[:, :, 3:19, 3:19, 3:19] = uf.to(dev)
        gb.gamer_refresh_ghosts_table(uf.to(dev), fine, nbr.to(dev))
        before = gb.gamer_launch_count()
        gb.gamer_interpolate_ghosts(c0.to(dev), fine, parent.to(dev), nbr.to(dev), coarse_in_new=c1.to(dev) if blend else None,
                                    w=0.25, monotonic=monotonic)
        torch.cuda.synchronize()
        assert gb.gamer_launch_count() == before + 1
        got = fine.cpu().double().numpy()
        if dtype == torch.float64:
            assert np.array_equal(got, ref)
        else:
            assert np.abs(got - ref).max() <= 1e-6 * np.abs(ref).max()
        keep = sibling_only != -7.0
        assert np.array_equal(got[keep], sibling_only[keep])


def test_config3_ghosts_filled_on_the_gpu(dev):
    """Config 3's fine-level preparation done entirely by the library (gamer_refresh_ghosts_table for siblings +
    gamer_interpolate_ghosts for the coarse-fine slabs, linear in time) equals the harness's global-array packing
    (amr.pack_fine) of the same two levels to round-off, at both sub-step times."""
    import amr_harness as amr
    uc, uf, region, dh_c = amr.sedov_two_level(32, 64, 64, gamma=G53, device=dev, e_blast=5.7e-5, p_amb=1.0)
    uc1 = uc * (1.0 + 0.05 * torch.sin(torch.arange(uc.shape[-1], device=dev) * 0.3))
    parent, _ = amr.region_tables(region, uc.shape[1:])
    nbr = amr.region_neighbors(region).to(dev)
    ug = amr.to_groups(uf)
    c0, c1 = inputs.pack_periodic(uc), inputs.pack_periodic(uc1)
    for w in (0.0, 0.5):
        ref, _ = amr.pack_fine(uf, (1.0 - w) * uc + w * uc1, region)
        fine = torch.zeros_like(ref)
        fine[:, :, 3:19, 3:19, 3:19] = ug
        gb.gamer_refresh_ghosts_table(ug, fine, nbr)
        gb.gamer_interpolate_ghosts(c0, fine, parent.to(dev), nbr, coarse_in_new=c1, w=w)
        torch.cuda.synchronize()
        assert (fine - ref).abs().max().item() <= 1e-14 * ref.abs().max().item()


def test_config3_step_with_library_preparation_and_fixup(dev):
    """One whole two-level step of config 3 (reduced size) in which every stage outside the harness's bookkeeping is a
    library call: sibling copy + coarse-fine interpolation in space and time for the fine level's ghosts, the solver, the
    restriction, flux averaging and flux correction.  Same result as the harness's own global-array preparation and fix-up
    to round-off, composite grid conserved to 1e-12."""
    import amr_harness as amr
    uc, uf, region, dh_c = amr.sedov_two_level(64, 128, 128, gamma=G53, device=dev)
    parent, _ = amr.region_tables(region, uc.shape[1:])
    parent, nbr = parent.to(dev), amr.region_neighbors(region).to(dev)
    z0, z1, y0, y1, x0, x1 = region
    fdims = ((z1 - z0) // 8, (y1 - y0) // 8, (x1 - x0) // 8)

    def gpu_solver(p, dt, dh):
        out, flux, speed, nun, diag = gpu_ex(p.contiguous(), dt, dh, G53, gb.MHM, gb.PLM, gb.HLLE, min_pres=1e-10)
        return out, flux

    def gpu_pack(uf_, uc0, uc1, w, region_):
        ug = amr.to_groups(uf_)
        fine = torch.empty((ug.shape[0], ug.shape[1], 22, 22, 22), dtype=ug.dtype, device=dev)
        fine[:, :, 3:19, 3:19, 3:19] = ug
        gb.gamer_refresh_ghosts_table(ug, fine, nbr)
        gb.gamer_interpolate_ghosts(inputs.pack_periodic(uc0), fine, parent, nbr, coarse_in_new=inputs.pack_periodic(uc1), w=w)
        return fine, fdims

    pb = (G53 - 1.0) / (8 * (0.5 * dh_c) ** 3)
    dt_c = 2 * 0.4 * (0.5 * dh_c) / (3.0 * math.sqrt(G53 * pb))
    tot0 = amr.composite_total(uc, uf, region, dh_c)
    ua, fa, _ = amr.two_level_step(gpu_solver, uc, uf, region, dh_c, dt_c)
    ub, fb, _ = amr.two_level_step(gpu_solver, uc, uf, region, dh_c, dt_c, fixup=_gpu_fixup(), pack_fine_fn=gpu_pack)
    torch.cuda.synchronize()
    for a, b in ((ua, ub), (fa, fb)):
        assert ((a - b).abs().amax(dim=(1, 2, 3)) <= 1e-12 * (a.abs().amax(dim=(1, 2, 3)) + 1e-30)).all()
    tot1 = amr.composite_total(ub, fb, region, dh_c)
    assert ((tot1 - tot0).abs() / (tot0.abs() + 1e-6)).max().item() <= 1e-12


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_poisson_sor_matches_oracle(dev, oracle_mod, dtype):
    """gamer_poisson_sor (R25) against oracle.poisson_sor on 37 patches (ragged against the
    148 SMs) of random potential guesses / boundary values and densities: after 1, 7 and 60 iterations the 18^3 potentials
    agree (fp64 1e-12, fp32 1e-5 of the scale), the outermost layer is untouched bit for bit, the acceleration of the 8^3
    active zones agrees, and 200 iterations reach the oracle's converged solution; acc = NULL and an empty batch work."""
    g = torch.Generator().manual_seed(9)
    n = 37
    phi0 = torch.randn((n, 18, 18, 18), generator=g, dtype=torch.float64).to(dtype)
    rho = (torch.randn((n, 16, 16, 16), generator=g, dtype=torch.float64) + 2.0).to(dtype)
    dh, coeff = 0.37, 4 * math.pi * 0.8
    omega = 2.0 / (1.0 + math.sin(math.pi / 17))
    tol = 1e-12 if dtype == torch.float64 else 1e-5
    edge = np.ones((18, 18, 18), bool)
    edge[1:17, 1:17, 1:17] = False
    for n_iter in (0, 1, 7, 60, 200):
        ref_phi, ref_acc = oracle_mod.poisson_sor(phi0.double().numpy(), rho.double().numpy(), dh, coeff, omega, n_iter)
        phi = phi0.to(dev).clone()
        acc = torch.full((n, 3, 8, 8, 8), float("nan"), dtype=dtype, device=dev)
        res = torch.full((n,), float("nan"), dtype=dtype, device=dev)
        gb.gamer_poisson_sor(phi, rho.to(dev), acc, dh, coeff, omega, n_iter, resid_out=res)
        torch.cuda.synchronize()
        got = phi.cpu().double().numpy()
        assert np.abs(got - ref_phi).max() <= tol * np.abs(ref_phi).max(), n_iter
        assert np.array_equal(got[:, edge], phi0.double().numpy()[:, edge])
        assert np.abs(acc.cpu().double().numpy() - ref_acc).max() <= 10 * tol * np.abs(ref_acc).max(), n_iter
        ref_res = oracle_mod.poisson_residual(ref_phi, rho.double().numpy(), dh, coeff)
        assert np.abs(res.cpu().double().numpy() - ref_res).max() <= 50 * tol * np.abs(ref_phi).max(), n_iter
        if n_iter == 200:
            assert res.max().item() <= 50 * tol * np.abs(ref_phi).max()        # converged: defect at round-off
    phi2 = phi0.to(dev).clone()
    gb.gamer_poisson_sor(phi2, rho.to(dev), None, dh, coeff, omega, 200)
    assert torch.equal(phi2, phi)                                     # acc = NULL: same potential, bitwise (run to run too)
    empty = torch.empty((0, 18, 18, 18), dtype=dtype, device=dev)
    gb.gamer_poisson_sor(empty, torch.empty((0, 16, 16, 16), dtype=dtype, device=dev), None, dh, coeff, omega, 5)


def _species_field(ns, n=32, seed=1712, entropy=False):
    """Mach-1 turbulence + ns species s_k = X_k rho (smooth positive X_k summing to one) [+ the entropy as last scalar]"""
    f = inputs.turbulence_field(n, seed, kmax=4, gamma=G53, entropy=entropy)
    rho = f[0]
    raw = [torch.exp(0.5 * inputs.random_field(rho.shape, seed + 31 * (k + 1), 4, "cpu")) for k in range(ns)]
    tot = sum(raw)
    spec = torch.stack([r / tot * rho for r in raw])
    return torch.cat([f[:5], spec, f[5:]], dim=0)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("ns", [2, 3, 4])
@pytest.mark.parametrize("scheme,recon,solver", [(gb.MHM, gb.PLM, gb.ROE), (gb.CTU, gb.PPM, gb.HLLC), (gb.VL, gb.PLM, gb.HLLC)])
def test_passive_scalars_match_oracle(dev, oracle_mod, scheme, recon, solver, ns, dtype):
    """N passive scalars, with and without renormalisation; ns = 3 also runs as 2 species + the entropy of
    the dual-energy formalism (the entropy is the last scalar and is not renormalised)."""
    for kw in (dict(), dict(renormalize=True)) + ((dict(renormalize=True, dual_energy=True),) if ns == 3 else ()):
        dual = bool(kw.get("dual_energy"))
        f = _species_field(ns - 1 if dual else ns, entropy=dual)
        padded = inputs.pack_periodic(f).to(dtype)
        p64 = padded.to(torch.float64)
        dh = 1 / 32
        dt = oracle_mod.cfl_dt(inputs.interior(p64).contiguous().numpy(), dh, G53, 0.4, scheme, oracle_mod.make_opts(n_scalar=ns))[0]
        ref = oracle_mod.fluid_advance(p64.numpy(), dt, dh, G53, scheme, recon, solver, oracle_mod.make_opts(n_scalar=ns, **kw))
        try:
            out, flux, speed, nun, diag = gpu_ex(padded.to(dev), dt, dh, G53, scheme, recon, solver, n_scalar=ns, **kw)
        except gb.GamerError as e:      # a tile that cannot fit in shared memory is refused, never computed wrongly
            assert "-2" in str(e) and dtype == torch.float64 and ns == 4, e
            continue
        tol = 1e-12 if dtype == torch.float64 else 1e-5
        err = rel_l1(out.cpu().numpy(), ref["out"], G53)
        assert max(err.values()) <= tol, (kw, err)
        o, r = out.cpu().numpy().astype(np.float64), ref["out"]
        for k in range(5, 5 + ns):
            assert np.abs(o[:, k] - r[:, k]).sum() <= tol * np.abs(r[:, k]).sum(), (kw, k)
        fe = np.abs(flux.cpu().numpy() - ref["flux"]).sum() / np.abs(ref["flux"]).sum()
        assert fe <= 2 * tol
        assert nun == ref["stats"]["n_unphysical"] == 0
        if kw.get("renormalize"):
            last = 5 + ns - (1 if dual else 0)
            ssum = o[:, 5:last].sum(axis=1)
            assert np.abs(ssum / o[:, 0] - 1.0).max() <= (1e-14 if dtype == torch.float64 else 1e-6)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("scheme,recon,solver,kw,dims", [
    (gb.MHM, gb.PLM, gb.ROE, {}, (2, 3, 4)),                                   # one ragged chunk
    (gb.CTU, gb.PPM, gb.HLLC, {}, (2, 3, 4)),
    (gb.VL, gb.PLM, gb.HLLC, dict(n_scalar=2, renormalize=True), (2, 3, 4)),
    (gb.MHM, gb.PLM, gb.HLLE, {}, (11, 10, 10)),                               # 1100 groups: two chunks, the second ragged
])
def test_host_entry_on_the_unpadded_state_is_bitwise_the_resident_entry(dev, scheme, recon, solver, kw, dims, dtype):
    """gamer_fluid_advance_host_resident: unpadded host state + host neighbour table in, host out / flux_out / speeds out,
    chunked copies overlapped with the fused-ghost kernels.  Must carry the bits of gamer_fluid_advance_resident on the
    whole batch (the same kernels on sub-ranges of the same device state), and of the padded host entry in fp64."""
    gz, gy, gx = dims
    ns = kw.get("n_scalar", 0)
    if gz * gy * gx > 100:
        gen = torch.Generator().manual_seed(5)
        rho = 1.0 + 0.3 * torch.rand((gz * 16, gy * 16, gx * 16), generator=gen, dtype=torch.float64)
        vel = [0.3 * (torch.rand(rho.shape, generator=gen, dtype=torch.float64) - 0.5) for _ in range(3)]
        f = inputs.prim_to_cons(rho, vel[0], vel[1], vel[2], torch.ones_like(rho), G53)
    else:
        f = _species_field(ns, n=16, seed=77)[:5 + ns] if ns else inputs.turbulence_field(16, 77, kmax=4, gamma=G53, shape=(gz * 16, gy * 16, gx * 16))
        if ns:
            f = torch.cat([f] * 1, dim=0)
            f = f.repeat(1, gz, gy, gx)
    padded = inputs.pack_periodic(f).to(dtype)
    u = inputs.interior(padded).contiguous()
    dt, dh = 0.002, 1.0 / 64
    nbr = gb.gamer_neighbors_periodic(gz, gy, gx, dev)
    ud = u.to(dev)
    out1, flux1, speed1 = gb.alloc_outputs(padded.to(dev))
    gb.gamer_fluid_advance_resident(ud, nbr, out1, flux1, dt, dh, G53, scheme, recon, solver, gb.make_opts(group_speed_out=speed1, **kw))
    torch.cuda.synchronize()
    h_u, h_nbr = u.pin_memory(), nbr.cpu().pin_memory()
    h_out, h_flux, h_speed = torch.empty_like(h_u).pin_memory(), torch.empty(flux1.shape, dtype=dtype).pin_memory(), torch.empty(speed1.shape, dtype=dtype).pin_memory()
    for _ in range(2):      # second call: scratch reused
        h_out.zero_()
        gb.gamer_fluid_advance_host_resident(h_u, h_nbr, h_out, h_flux, h_speed, dt, dh, G53, scheme, recon, solver,
                                             gb.make_opts(on_device=False, **kw))
        assert torch.equal(h_out, out1.cpu()) and torch.equal(h_flux, flux1.cpu()) and torch.equal(h_speed, speed1.cpu())
    if dtype == torch.float64 and not kw:
        p_out, p_flux, p_speed = torch.empty_like(h_out), torch.empty_like(h_flux), torch.empty_like(h_speed)
        gb.gamer_fluid_advance_host(padded.contiguous(), p_out, p_flux, p_speed, dt, dh, G53, scheme, recon, solver)
        assert (p_out - h_out).abs().max().item() <= 1e-13 * h_out.abs().max().item()
    # bad table entries and unsupported options are refused before any copy
    bad = h_nbr.clone()
    bad[0, 5] = gz * gy * gx
    with pytest.raises(gb.GamerError, match="-1"):
        gb.gamer_fluid_advance_host_resident(h_u, bad, h_out, h_flux, h_speed, dt, dh, G53, scheme, recon, solver, gb.make_opts(on_device=False, **kw))
    with pytest.raises(gb.GamerError):      # the binding's own shape check catches it before the C entry would (-1)
        gb.gamer_fluid_advance_host_resident(h_u, h_nbr, h_out, h_flux, h_speed, dt, dh, G53, scheme, recon, solver, gb.make_opts(on_device=False, n_scalar=7))
    with pytest.raises(gb.GamerError, match="-2"):
        gb.gamer_fluid_advance_host_resident(h_u, h_nbr, h_out, h_flux, h_speed, dt, dh, G53, scheme, recon, solver,
                                             gb.make_opts(on_device=False, remedy_first_order=True, **kw))
    gb.gamer_release_scratch()


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_gravity_update_fused_and_standalone_match_oracle(dev, oracle_mod, dtype):
    """the fluid's gravity update right behind the Poisson solve.  gamer_poisson_sor_gravity (fused: the
    acceleration never leaves the SM) and gamer_poisson_sor + gamer_gravity_update must both equal the oracle's
    poisson_sor -> gravity_update composition; group 1's octants are checked against the patch numbering."""
    gen = torch.Generator().manual_seed(12)
    ng, nv = 3, 6
    npatch = 8 * ng
    phi = torch.randn((npatch, 18, 18, 18), generator=gen, dtype=torch.float64)
    rho_p = torch.rand((npatch, 16, 16, 16), generator=gen, dtype=torch.float64) + 0.5
    flu = torch.empty((ng, nv, 16, 16, 16), dtype=torch.float64)
    flu[:, 0] = torch.rand((ng, 16, 16, 16), generator=gen, dtype=torch.float64) + 0.5
    flu[:, 1:4] = flu[:, 0:1] * 0.4 * torch.randn((ng, 3, 16, 16, 16), generator=gen, dtype=torch.float64)
    flu[:, 4] = 1.5 + 0.5 * (flu[:, 1:4] ** 2).sum(dim=1) / flu[:, 0]
    flu[:, 5] = torch.rand((ng, 16, 16, 16), generator=gen, dtype=torch.float64)
    phi, rho_p, flu = phi.to(dtype), rho_p.to(dtype), flu.to(dtype)
    dh, coeff, om, nit, dt = 0.1, 1.3, 1.6, 12, 0.07
    rphi, racc = oracle_mod.poisson_sor(phi.double().numpy(), rho_p.double().numpy(), dh, coeff, om, nit)
    ref = oracle_mod.gravity_update(flu.double().numpy(), racc, dt)
    tol = 1e-13 if dtype == torch.float64 else 2e-5
    # fused
    p1, f1 = phi.clone().to(dev), flu.clone().to(dev)
    acc1 = torch.empty((npatch, 3, 8, 8, 8), dtype=dtype, device=dev)
    gb.gamer_poisson_sor_gravity(p1, rho_p.to(dev), acc1, f1, dt, dh, coeff, om, nit)
    # two calls
    p2, f2 = phi.clone().to(dev), flu.clone().to(dev)
    acc2 = torch.empty_like(acc1)
    gb.gamer_poisson_sor(p2, rho_p.to(dev), acc2, dh, coeff, om, nit)
    gb.gamer_gravity_update(f2, acc2, dt)
    # fused without the acceleration output
    p3, f3 = phi.clone().to(dev), flu.clone().to(dev)
    gb.gamer_poisson_sor_gravity(p3, rho_p.to(dev), None, f3, dt, dh, coeff, om, nit)
    torch.cuda.synchronize()
    assert torch.equal(p1, p2) and torch.equal(acc1, acc2) and torch.equal(f1, f2) and torch.equal(f1, f3)
    scale = np.abs(ref).max(axis=(0, 2, 3, 4), keepdims=True)
    assert (np.abs(f1.cpu().numpy() - ref) / scale).max() <= tol
    assert torch.equal(f1[:, 0], flu[:, 0].to(dev)) and torch.equal(f1[:, 5], flu[:, 5].to(dev))      # density, scalar untouched
    assert (f1[:, 1:5] - flu[:, 1:5].to(dev)).abs().max().item() > 1e-3
    # a kick and its opposite
    gb.gamer_gravity_update(f2, acc2, -dt)
    torch.cuda.synchronize()
    assert ((f2.cpu() - flu).abs().max().item()) <= (1e-13 if dtype == torch.float64 else 1e-5) * flu.abs().max().item()
    # n_patches must be whole groups
    with pytest.raises(gb.GamerError):
        gb.gamer_gravity_update(f2, acc2[:7].contiguous(), dt)
