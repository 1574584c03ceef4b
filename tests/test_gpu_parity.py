"""GPU parity: the CUDA path (through the C ABI) against the fp64 CPU oracle, element by element on the
same seeded inputs.  Tolerances are BASELINE.json's: fp64 relative L1 <= 1e-12 per step; fp32 <= 1e-5
per step and <= 1e-4 after 10 steps.  Norms: tests/helpers.rel_l1."""
import itertools
import math

import numpy as np
import pytest
import torch

from helpers import rel_l1
from paper_1712_07070_b200 import binding as gb
from paper_1712_07070_b200 import inputs

pytestmark = pytest.mark.gpu

G53 = 5.0 / 3.0
TOL = {torch.float64: 1e-12, torch.float32: 1e-5}
SCHEMES = [gb.MHM, gb.CTU]
COMBOS = list(itertools.product(SCHEMES, (gb.PLM, gb.PPM), (gb.ROE, gb.HLLC, gb.HLLE))) + \
    [(gb.MHM, gb.PLM, gb.EXACT), (gb.CTU, gb.PPM, gb.EXACT), (gb.MHM, gb.PPM, gb.EXACT), (gb.CTU, gb.PLM, gb.EXACT)] + \
    [(gb.VL, gb.PLM, s) for s in (gb.ROE, gb.HLLC, gb.HLLE, gb.EXACT)]      # VL scheme, PLM only


@pytest.fixture(scope="module")
def dev():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    gb.lib()
    return torch.device("cuda:0")


def flux_err(a, b, gamma):
    """relative L1 of flux_out [G,3,3,NV,16,16] per variable class, normalised by sum|F| of that class."""
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
    out = {}
    out["mass"] = np.abs(a[:, :, :, 0] - b[:, :, :, 0]).sum() / max(np.abs(b[:, :, :, 0]).sum(), 1e-300)
    out["mom"] = np.abs(a[:, :, :, 1:4] - b[:, :, :, 1:4]).sum() / max(np.abs(b[:, :, :, 1:4]).sum(), 1e-300)
    out["ener"] = np.abs(a[:, :, :, 4] - b[:, :, :, 4]).sum() / max(np.abs(b[:, :, :, 4]).sum(), 1e-300)
    return out


def run_gpu(padded, dt, dh, gamma, scheme, recon, solver, opts_kw=None, use_ex=True):
    out, flux, speed = gb.alloc_outputs(padded)
    if use_ex:
        o = gb.make_opts(group_speed_out=speed, **(opts_kw or {}))
        gb.gamer_fluid_advance_ex(padded, out, flux, dt, dh, gamma, scheme, recon, solver, o)
    else:
        gb.gamer_fluid_advance(padded, out, flux, dt, dh, gamma, scheme, recon, solver)
    torch.cuda.synchronize()
    return out, flux, speed


def oracle_dt(oracle, padded64, dh, gamma, cfl, scheme):
    return oracle.cfl_dt(inputs.interior(padded64).contiguous().numpy(), dh, gamma, cfl, scheme)[0]


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("scheme,recon,solver", COMBOS)
def test_one_step_matches_oracle(dev, oracle_mod, scheme, recon, solver, dtype):
    """48^3 Mach-1 turbulence = 27 groups (several tiles per SM wave and a ragged last wave)."""
    f = inputs.turbulence_field(48, 1712, kmax=4, gamma=G53)
    padded = inputs.pack_periodic(f).to(dtype)                 # rounded to the run precision
    p64 = padded.to(torch.float64)                             # the oracle sees the same rounded values
    dh = 1.0 / 48
    dt = oracle_dt(oracle_mod, p64, dh, G53, 0.4, scheme)
    ref = oracle_mod.fluid_advance(p64.numpy(), dt, dh, G53, scheme, recon, solver)
    out, flux, speed = run_gpu(padded.to(dev), dt, dh, G53, scheme, recon, solver)
    tol = TOL[dtype]
    err = rel_l1(out.cpu().numpy(), ref["out"], G53)
    assert max(err.values()) <= tol, err
    ferr = flux_err(flux.cpu().numpy(), ref["flux"], G53)
    assert max(ferr.values()) <= 2 * tol, ferr
    serr = np.abs(speed.cpu().numpy() - ref["speed"]).max() / ref["speed"].max()
    assert serr <= (1e-12 if dtype == torch.float64 else 2e-6), serr
    if dtype == torch.float64:
        # element-wise too, not only in the norm
        scale = np.abs(ref["out"]).max(axis=(0, 2, 3, 4), keepdims=True)
        assert (np.abs(out.cpu().numpy() - ref["out"]) / scale).max() <= 1e-11


@pytest.mark.parametrize("scheme,recon,solver", [(gb.MHM, gb.PLM, gb.ROE), (gb.CTU, gb.PPM, gb.HLLC), (gb.VL, gb.PLM, gb.HLLC)])
def test_fp64_is_bitwise_reproducible_and_eleven_arg_form_agrees(dev, scheme, recon, solver):
    """bitwise reproducibility (run to run)."""
    f = inputs.turbulence_field(32, 7, kmax=4, gamma=G53)
    padded = inputs.pack_periodic(f).to(dev)
    a = run_gpu(padded, 0.003, 1 / 32, G53, scheme, recon, solver)
    b = run_gpu(padded, 0.003, 1 / 32, G53, scheme, recon, solver)
    c = run_gpu(padded, 0.003, 1 / 32, G53, scheme, recon, solver, use_ex=False)
    for x, y in zip(a, b):
        assert torch.equal(x, y)
    assert torch.equal(a[0], c[0]) and torch.equal(a[1], c[1])


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("scheme,recon,solver", COMBOS)
def test_uniform_state_bitwise_invariant(dev, scheme, recon, solver, dtype):
    one = torch.ones((16, 16, 16), dtype=torch.float64)
    f = inputs.prim_to_cons(1.3 * one, 0.7 * one, -0.45 * one, 0.3 * one, 0.9 * one, G53)
    padded = inputs.pack_periodic(f).to(dtype).to(dev)
    out, _, _ = run_gpu(padded, 0.01, 1 / 16, G53, scheme, recon, solver)
    assert torch.equal(out, inputs.interior(padded))


@pytest.mark.parametrize("scheme,recon,solver", [(gb.MHM, gb.PLM, gb.ROE), (gb.CTU, gb.PPM, gb.HLLC), (gb.VL, gb.PLM, gb.ROE)])
def test_shared_faces_bitwise_equal_and_conservation(dev, scheme, recon, solver):
    f = inputs.turbulence_field(32, 1712, kmax=4, gamma=G53)
    padded = inputs.pack_periodic(f).to(dev)
    out, flux, _ = run_gpu(padded, 0.003, 1 / 32, G53, scheme, recon, solver)
    fl = flux.cpu().numpy().reshape(2, 2, 2, 3, 3, 5, 16, 16)
    for gz, gy, gx in itertools.product(range(2), repeat=3):
        assert np.array_equal(fl[gz, gy, gx, 0, 2], fl[gz, gy, (gx + 1) % 2, 0, 0])
        assert np.array_equal(fl[gz, gy, gx, 1, 2], fl[gz, (gy + 1) % 2, gx, 1, 0])
        assert np.array_equal(fl[gz, gy, gx, 2, 2], fl[(gz + 1) % 2, gy, gx, 2, 0])
    new = inputs.unpack(out.cpu(), 2, 2, 2)
    for v in range(5):
        s0, s1 = math.fsum(f[v].flatten().tolist()), math.fsum(new[v].flatten().tolist())
        assert abs(s1 - s0) <= 1e-13 * (math.fsum(f[v].abs().flatten().tolist()) + 1.0)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_config1_sod_ten_steps_device_resident_loop(dev, oracle_mod, dtype):
    """BASELINE.json config 1: 64^3 Sod, MHM+PLM(minmod)+Roe, CFL 0.5, 10 steps; the GPU loop is
    advance -> cfl_dt (device dt) -> periodic ghost refresh, all on the device; the oracle loop repacks on
    the host.  fp32 must stay within 1e-5 per step (restarted from the oracle state) and 1e-4 after 10."""
    gamma, dh, n = 1.4, 1.0 / 64, 64
    f = inputs.sod_field(n, gamma)
    padded = inputs.pack_periodic(f).to(dtype)
    u_or = padded.to(torch.float64)
    u_gpu = padded.to(dev)
    out, flux, speed = gb.alloc_outputs(u_gpu)
    dt_dev = torch.zeros(1, dtype=torch.float64, device=dev)
    gb.gamer_cfl_dt(inputs.interior(u_gpu).contiguous(), dh, gamma, 0.5, gb.MHM, None, dt_dev)
    tol1, tol10 = (1e-12, 1e-11) if dtype == torch.float64 else (1e-5, 1e-4)
    for step in range(10):
        dt_or = oracle_dt(oracle_mod, u_or, dh, gamma, 0.5, gb.MHM)
        torch.cuda.synchronize()
        assert abs(dt_dev.item() - dt_or) <= (1e-13 if dtype == torch.float64 else 1e-5) * dt_or
        ref = oracle_mod.fluid_advance(u_or.numpy(), dt_or, dh, gamma, gb.MHM, gb.PLM, gb.ROE, want_flux=False)
        o = gb.make_opts(dt_dev=dt_dev, group_speed_out=speed)
        gb.gamer_fluid_advance_ex(u_gpu, out, flux, 1.0, dh, gamma, gb.MHM, gb.PLM, gb.ROE, o)
        gb.gamer_cfl_from_group_speed(speed, dh, 0.5, dt_dev)
        # per-step error: same step from the oracle's state rounded to the run precision
        o1 = gb.alloc_outputs(u_gpu, want_flux=False, want_speed=False)[0]
        gb.gamer_fluid_advance_ex(u_or.to(dtype).to(dev), o1, None, dt_or, dh, gamma, gb.MHM, gb.PLM, gb.ROE,
                                  gb.make_opts())
        ref_in = oracle_mod.fluid_advance(u_or.to(dtype).to(torch.float64).numpy(), dt_or, dh, gamma, gb.MHM, gb.PLM,
                                          gb.ROE, want_flux=False)
        e1 = rel_l1(o1.cpu().numpy(), ref_in["out"], gamma)
        assert max(e1.values()) <= tol1, (step, e1)
        gb.gamer_refresh_ghosts_periodic(out, u_gpu, 4, 4, 4)
        u_or = inputs.pack_periodic(inputs.unpack(torch.from_numpy(ref["out"]), 4, 4, 4))
    torch.cuda.synchronize()
    e10 = rel_l1(inputs.interior(u_gpu).cpu().numpy(), inputs.interior(u_or).numpy(), gamma)
    assert max(e10.values()) <= tol10, e10
    # conservation over the 10 steps on the GPU side (fp64: round-off; fp32: accumulated rounding)
    tot0 = f.sum(dim=(1, 2, 3))
    tot1 = inputs.unpack(inputs.interior(u_gpu).cpu().to(torch.float64).contiguous(), 4, 4, 4).sum(dim=(1, 2, 3))
    assert abs(tot1[0] - tot0[0]) <= (1e-12 if dtype == torch.float64 else 2e-6) * tot0[0]


def test_ghost_refresh_matches_host_packing(dev):
    f = inputs.turbulence_field(32, 5, kmax=3, gamma=G53, shape=(48, 32, 64), entropy=True)
    padded = inputs.pack_periodic(f)
    u = inputs.interior(padded).contiguous().to(dev)
    got = torch.empty_like(padded, device=dev)
    gb.gamer_refresh_ghosts_periodic(u, got, 3, 2, 4)
    torch.cuda.synchronize()
    assert torch.equal(got.cpu(), padded)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_cfl_dt_matches_oracle(dev, oracle_mod, dtype):
    f = inputs.turbulence_field(32, 11, kmax=4, gamma=G53)
    u = inputs.interior(inputs.pack_periodic(f)).contiguous().to(dtype)
    for scheme in (gb.MHM, gb.CTU):
        dt_ref, sp_ref = oracle_mod.cfl_dt(u.to(torch.float64).numpy(), 1 / 32, G53, 0.5, scheme)
        sp = torch.empty(u.shape[0], dtype=dtype, device=dev)
        dt = torch.zeros(1, dtype=torch.float64, device=dev)
        gb.gamer_cfl_dt(u.to(dev), 1 / 32, G53, 0.5, scheme, sp, dt)
        torch.cuda.synchronize()
        tol = 1e-13 if dtype == torch.float64 else 2e-6
        assert np.abs(sp.cpu().numpy() - sp_ref).max() <= tol * sp_ref.max()
        assert abs(dt.item() - dt_ref) <= tol * dt_ref


def test_empty_batch_is_a_noop(dev):
    z = torch.empty((0, 5, 22, 22, 22), dtype=torch.float32, device=dev)
    out, flux, speed = gb.alloc_outputs(z)
    gb.gamer_fluid_advance(z, out, flux, 0.1, 0.1, 1.4, gb.MHM, gb.PLM, gb.ROE)
    torch.cuda.synchronize()


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("scheme,recon,solver", [(gb.MHM, gb.PLM, gb.ROE), (gb.CTU, gb.PPM, gb.HLLC)])
def test_ragged_batches_and_host_entry_agree_bitwise(dev, scheme, recon, solver, dtype):
    """Groups are independent: any batch size (1, a prime, a size that is not a multiple of the host entry's chunk)
    gives the same bits per group as the full batch, and the host-buffer entry (gamer_fluid_advance_host, the
    e2e path of bench.py: chunked H2D -> kernel -> D2H) gives the same bits as the device entry."""
    f = inputs.turbulence_field(144, 99, kmax=6, gamma=G53)            # 9^3 = 729 groups > one 592-group chunk
    padded = inputs.pack_periodic(f).to(dtype)
    dt, dh = 0.3 / 144 / 4.0, 1.0 / 144
    full = run_gpu(padded.to(dev), dt, dh, G53, scheme, recon, solver)
    for n in (1, 37):
        part = run_gpu(padded[:n].contiguous().to(dev), dt, dh, G53, scheme, recon, solver)
        for a, b in zip(part, full):
            assert torch.equal(a, b[:n])
    h_in = padded.contiguous().pin_memory()
    h_out = torch.empty(tuple(full[0].shape), dtype=dtype).pin_memory()
    h_flux = torch.empty(tuple(full[1].shape), dtype=dtype).pin_memory()
    h_speed = torch.empty(tuple(full[2].shape), dtype=dtype).pin_memory()
    gb.gamer_fluid_advance_host(h_in, h_out, h_flux, h_speed, dt, dh, G53, scheme, recon, solver)
    assert torch.equal(h_out, full[0].cpu()) and torch.equal(h_flux, full[1].cpu()) and torch.equal(h_speed, full[2].cpu())
    assert torch.isfinite(h_out).all()


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("scheme,recon,solver", [(gb.MHM, gb.PLM, gb.ROE), (gb.MHM, gb.PPM, gb.HLLC), (gb.CTU, gb.PPM, gb.HLLC),
                                                 (gb.CTU, gb.PLM, gb.HLLE)])
def test_repeated_launches_on_a_busy_gpu_are_bitwise_identical(dev, scheme, recon, solver, dtype):
    """Run-to-run reproducibility under load: 1728 groups (more CTAs than fit on the GPU at once, so
    CTAs of different planes and groups overlap in every order), five launches, every output identical bit for bit.
    The kernels exchange face states and fluxes through double-buffered shared memory with one barrier per plane; a
    missing barrier or a buffer reused one plane too early shows up here as a difference between launches."""
    f = inputs.turbulence_field(192, 31, kmax=8, gamma=G53, device=dev)
    padded = inputs.pack_periodic(f, dtype=dtype)
    dt, dh = 0.25 / 192 / 4.0, 1.0 / 192
    first = run_gpu(padded, dt, dh, G53, scheme, recon, solver)
    assert torch.isfinite(first[0]).all()
    for _ in range(4):
        again = run_gpu(padded, dt, dh, G53, scheme, recon, solver)
        for x, y in zip(first, again):
            assert torch.equal(x, y)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_ghost_refresh_with_boundary_conditions_matches_oracle(dev, oracle_mod, dtype):
    """gamer_refresh_ghosts (PAPER.md L98 boundary conditions, L248 preparation) against oracle.fill_ghosts, bit for
    bit: outflow / reflecting / periodic mixed over the six faces, 5 and 6 variables (the scalar never changes sign)."""
    O, R, P = gb.BC_OUTFLOW, gb.BC_REFLECTING, gb.BC_PERIODIC
    for nv in (5, 6):
        f = inputs.turbulence_field(16, 77, kmax=4, gamma=G53, shape=(32, 48, 16), entropy=(nv == 6)).to(dtype)
        u = inputs.interior(inputs.pack_periodic(f)).contiguous().to(dev)
        for bc in ((O, R, R, O, P, P), (R, R, P, P, O, R), (P, P, P, P, P, P)):
            ref = oracle_mod.fill_ghosts(f.numpy(), ((bc[0], bc[1]), (bc[2], bc[3]), (bc[4], bc[5])))
            padded = torch.full((u.shape[0], nv, 22, 22, 22), float("nan"), dtype=dtype, device=dev)
            gb.gamer_refresh_ghosts(u, padded, 2, 3, 1, bc)
            torch.cuda.synchronize()
            assert np.array_equal(padded.cpu().numpy(), ref)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_config1_sod_with_outflow_in_x_as_stated(dev, oracle_mod, dtype):
    """BASELINE.json config 1 as worded -- "periodic-in-y/z": the tube is open along x (outflow), periodic in y and z.
    Same device-resident loop as above with gamer_refresh_ghosts; the oracle loop refills with oracle.fill_ghosts.
    (The fully periodic variant above is the one SURVEY 8(d) specifies; this one needs the L98 boundary fill.)"""
    gamma, dh, n = 1.4, 1.0 / 64, 64
    f = inputs.sod_field(n, gamma)
    bc = (gb.BC_OUTFLOW, gb.BC_OUTFLOW, gb.BC_PERIODIC, gb.BC_PERIODIC, gb.BC_PERIODIC, gb.BC_PERIODIC)
    obc = ((oracle_mod.OUTFLOW, oracle_mod.OUTFLOW), (oracle_mod.PERIODIC,) * 2, (oracle_mod.PERIODIC,) * 2)
    u_or = torch.from_numpy(oracle_mod.fill_ghosts(f.to(dtype).to(torch.float64).numpy(), obc))
    state = inputs.interior(inputs.pack_periodic(f)).contiguous().to(dtype).to(dev)
    u_gpu = torch.empty((64, 5, 22, 22, 22), dtype=dtype, device=dev)
    gb.gamer_refresh_ghosts(state, u_gpu, 4, 4, 4, bc)
    out, flux, speed = gb.alloc_outputs(u_gpu)
    dt_dev = torch.zeros(1, dtype=torch.float64, device=dev)
    gb.gamer_cfl_dt(state, dh, gamma, 0.5, gb.MHM, None, dt_dev)
    for step in range(10):
        dt_or = oracle_dt(oracle_mod, u_or, dh, gamma, 0.5, gb.MHM)
        ref = oracle_mod.fluid_advance(u_or.numpy(), dt_or, dh, gamma, gb.MHM, gb.PLM, gb.ROE, want_flux=False)
        gb.gamer_fluid_advance_ex(u_gpu, out, flux, 1.0, dh, gamma, gb.MHM, gb.PLM, gb.ROE,
                                  gb.make_opts(dt_dev=dt_dev, group_speed_out=speed))
        gb.gamer_cfl_from_group_speed(speed, dh, 0.5, dt_dev)
        gb.gamer_refresh_ghosts(out, u_gpu, 4, 4, 4, bc)
        u_or = torch.from_numpy(oracle_mod.fill_ghosts(inputs.unpack(torch.from_numpy(ref["out"]), 4, 4, 4).numpy(), obc))
    torch.cuda.synchronize()
    e10 = rel_l1(inputs.interior(u_gpu).cpu().numpy(), inputs.interior(u_or).numpy(), gamma)
    assert max(e10.values()) <= (1e-11 if dtype == torch.float64 else 1e-4), e10
    # the tube stayed one-dimensional and nothing reached the open ends yet: the end states are the initial ones
    new = inputs.unpack(inputs.interior(u_gpu).cpu().to(torch.float64).contiguous(), 4, 4, 4)
    assert (new[0, :, :, 0] - 1.0).abs().max() <= 1e-6 and (new[0, :, :, -1] - 0.125).abs().max() <= 1e-6
    assert (new[0] - new[0, :1, :1, :]).abs().max() <= 1e-6


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_table_driven_ghost_refresh_matches_oracle(dev, oracle_mod, dtype):
    """gamer_refresh_ghosts_table (sibling copy of L248 for any same-level topology) against oracle.fill_ghosts_table,
    bit for bit, including slabs without a same-level neighbour (-1), which must keep their previous content."""
    f = inputs.turbulence_field(16, 5, kmax=4, gamma=G53, shape=(32, 48, 16)).to(dtype)
    u = inputs.interior(inputs.pack_periodic(f)).contiguous()
    nbr = gb.gamer_neighbors_periodic(2, 3, 1, dev).cpu()
    nbr[:, 14] = -1
    nbr[3, 4] = -1
    nbr[5, 0] = -1
    before = torch.randn((6, 5, 22, 22, 22), generator=torch.Generator().manual_seed(1), dtype=torch.float64).to(dtype)
    ref = oracle_mod.fill_ghosts_table(u.numpy(), nbr.numpy(), before.numpy().copy())
    padded = before.to(dev).clone()
    gb.gamer_refresh_ghosts_table(u.to(dev), padded, nbr.to(dev))
    torch.cuda.synchronize()
    assert np.array_equal(padded.cpu().numpy(), ref)
    assert not np.array_equal(ref, before.numpy())


def test_vl_with_ppm_is_unsupported(dev):
    """VL + PPM would read a fourth ghost zone; the header promises GAMER_EUNSUPPORTED."""
    padded = inputs.pack_periodic(inputs.turbulence_field(16, 3, kmax=2, gamma=G53)).to(dev)
    out, flux, _ = gb.alloc_outputs(padded)
    with pytest.raises(gb.GamerError, match="-2"):
        gb.gamer_fluid_advance(padded, out, flux, 1e-3, 1 / 16, G53, gb.VL, gb.PPM, gb.ROE)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_paper_kelvin_helmholtz_workload(dev, oracle_mod, dtype):
    """The paper's own uniform-grid workload (shear layers of density 2 / 1 and v_x = +-0.5, P = 2.5, gamma = 1.4,
    white-noise velocity perturbation of 1e-2) with the scheme it was run with, CTU + PPM + Roe (L338), on 64^3 cells = 64
    groups: three device-resident steps (advance, dt from the fused CFL maxima, periodic ghost refresh) against the oracle
    stepping the same way.  Discontinuous data + noise: every limiter branch is exercised."""
    n, gamma, cfl = 64, 1.4, 0.4
    f = inputs.kh_field(n, gamma=gamma)
    dh = 1.0 / n
    gz = gy = gx = n // 16
    padded = inputs.pack_periodic(f).to(dtype)
    u_in = padded.to(dev)
    out, flux, speed = gb.alloc_outputs(u_in)
    dt_dev = torch.zeros(1, dtype=torch.float64, device=dev)
    gb.gamer_cfl_dt(inputs.interior(u_in).contiguous(), dh, gamma, cfl, gb.CTU, None, dt_dev)
    opts = gb.make_opts(dt_dev=dt_dev, group_speed_out=speed)
    ref = padded.to(torch.float64)
    tol = 1e-12 if dtype == torch.float64 else 1e-5
    for step in range(3):
        dt_ref, _ = oracle_mod.cfl_dt(inputs.interior(ref).contiguous().numpy(), dh, gamma, cfl, gb.CTU)
        r = oracle_mod.fluid_advance(ref.numpy(), dt_ref, dh, gamma, gb.CTU, gb.PPM, gb.ROE, want_flux=False)
        gb.gamer_fluid_advance_ex(u_in, out, flux, 1.0, dh, gamma, gb.CTU, gb.PPM, gb.ROE, opts)
        dt_gpu = float(dt_dev.item())
        assert abs(dt_gpu - dt_ref) <= (1e-12 if dtype == torch.float64 else 2e-6) * dt_ref * (step + 1)
        err = rel_l1(out.cpu().numpy(), r["out"], gamma)
        assert max(err.values()) <= tol * (step + 1), (step, err)
        gb.gamer_cfl_from_group_speed(speed, dh, cfl, dt_dev)
        gb.gamer_refresh_ghosts_periodic(out, u_in, gz, gy, gx)
        ref = inputs.pack_periodic(inputs.unpack(torch.from_numpy(r["out"]), gz, gy, gx))
    torch.cuda.synchronize()
    assert torch.isfinite(out).all()
    # mass and x momentum of the periodic box are conserved over the three steps
    new = inputs.unpack(out.cpu().to(torch.float64), gz, gy, gx)
    for v in (0, 1, 4):
        s0, s1 = f[v].sum().item(), new[v].sum().item()
        assert abs(s1 - s0) <= (1e-12 if dtype == torch.float64 else 3e-6) * f[v].abs().sum().item()
