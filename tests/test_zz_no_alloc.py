"""gamer_fluid_advance_table_noalloc: the allocation-free entry (static 64 MiB device scratch instead of a caller-allocated
padded batch) against the existing path it mirrors, gamer_refresh_ghosts_table + gamer_fluid_advance_ex.  Collected last on
purpose (file name): the suite runs with pytest -x, a failure here must not hide other tests."""
import ctypes

import pytest
import torch

from paper_1712_07070_b200 import binding as gb
from paper_1712_07070_b200 import inputs

pytestmark = pytest.mark.gpu
G53 = 5.0 / 3.0


@pytest.fixture(scope="module")
def dev():
    assert torch.cuda.is_available()
    gb.lib()
    return torch.device("cuda:0")


def _existing_path(u, nbr, dt, dh, scheme, recon, solver, kw):
    """caller-allocated padded batch -> sibling copy -> padded kernel"""
    g, nv = u.shape[:2]
    padded = torch.zeros((g, nv, 22, 22, 22), dtype=u.dtype, device=u.device)
    gb.gamer_refresh_ghosts_table(u, padded, nbr)
    out, flux, speed = gb.alloc_outputs(padded)
    nun = torch.zeros(1, dtype=torch.int32, device=u.device)
    gb.gamer_fluid_advance_ex(padded, out, flux, dt, dh, G53, scheme, recon, solver,
                              gb.make_opts(group_speed_out=speed, n_unphysical_out=nun, **kw))
    torch.cuda.synchronize()
    return out, flux, speed, nun


def _noalloc(u, nbr, dt, dh, scheme, recon, solver, kw, out, flux, speed, nun):
    gb.gamer_fluid_advance_table_noalloc(u, nbr, out, flux, dt, dh, G53, scheme, recon, solver,
                                         gb.make_opts(group_speed_out=speed, n_unphysical_out=nun, **kw))
    torch.cuda.synchronize()


@pytest.mark.parametrize("dtype", [torch.float32, torch.float64])
def test_noalloc_entry_equals_refresh_plus_advance_on_two_calls_in_a_row(dev, dtype):
    """Two calls in a row on DIFFERENT batches (the second smaller, so stale contents of the shared array would show), each
    against refresh + advance with a caller-allocated padded batch.  Same kernels on the same values: the tests' tolerance for
    this pair is bitwise equality.  The second call also runs remedy (ii), which needs the padded slab in memory."""
    cases = [((2, 3, 4), gb.MHM, gb.PLM, gb.ROE, {}, 1.0, 1.0),
             ((2, 2, 2), gb.CTU, gb.PPM, gb.HLLC, dict(remedy_first_order=True), 6.0, 2.0)]
    outs = []
    for (gz, gy, gx), scheme, recon, solver, kw, mach, sigma in cases:
        f = inputs.turbulence_field(16, 4242 + gz, kmax=4, gamma=G53, shape=(gz * 16, gy * 16, gx * 16), mach=mach, sigma=sigma)
        u = inputs.interior(inputs.pack_periodic(f)).contiguous().to(dtype).to(dev)
        nbr = gb.gamer_neighbors_periodic(gz, gy, gx, dev)
        dt, dh = 0.003 / mach, 1.0 / 64
        ref = _existing_path(u, nbr, dt, dh, scheme, recon, solver, kw)
        out, flux, speed = (torch.full_like(t, float("nan")) for t in ref[:3])
        nun = torch.full((1,), -1, dtype=torch.int32, device=dev)
        _noalloc(u, nbr, dt, dh, scheme, recon, solver, kw, out, flux, speed, nun)
        assert torch.isfinite(out).all()
        assert torch.equal(out, ref[0]) and torch.equal(flux, ref[1]) and torch.equal(speed, ref[2]) and torch.equal(nun, ref[3])
        outs.append((u, nbr, dt, dh, scheme, recon, solver, kw, ref))
    # and the first batch once more after the second: the shared array carries nothing over
    u, nbr, dt, dh, scheme, recon, solver, kw, ref = outs[0]
    out, flux, speed = (torch.empty_like(t) for t in ref[:3])
    nun = torch.zeros(1, dtype=torch.int32, device=dev)
    _noalloc(u, nbr, dt, dh, scheme, recon, solver, kw, out, flux, speed, nun)
    assert torch.equal(out, ref[0]) and torch.equal(flux, ref[1]) and torch.equal(speed, ref[2])


def test_noalloc_entry_limits_and_allocates_nothing(dev):
    """Sizes beyond the static array are refused with GAMER_ETOOLARGE before anything is enqueued; device memory in use
    (cudaMemGetInfo) does not move across calls."""
    assert gb.gamer_noalloc_max_groups(5, gb.FP32) == (64 << 20) // (5 * 22 ** 3 * 4) == 315
    assert gb.gamer_noalloc_max_groups(5, gb.FP64) == 157 and gb.gamer_noalloc_max_groups(9, gb.FP64) == 87
    assert gb.gamer_noalloc_max_groups(4, gb.FP32) == 0 and gb.gamer_noalloc_max_groups(5, 2) == 0
    L = gb.lib()
    vp = ctypes.c_void_p
    big = gb.gamer_noalloc_max_groups(5, gb.FP32) + 1
    assert L.gamer_fluid_advance_table_noalloc(vp(4096), vp(8192), vp(16384), None, big, 0.1, 0.1, 1.4, 1, 1, 1, 4, None) == -5
    assert b"static scratch" in L.gamer_strerror(-5)
    assert L.gamer_fluid_advance_table_noalloc(vp(4096), vp(8192), vp(16384), None, 0, 0.1, 0.1, 1.4, 1, 1, 1, 4, None) == 0
    assert L.gamer_fluid_advance_table_noalloc(None, vp(8192), vp(16384), None, 1, 0.1, 0.1, 1.4, 1, 1, 1, 4, None) == -1
    # the largest batch that fits, three times: free device memory unchanged
    g = 315
    gen = torch.Generator().manual_seed(1)
    rho = 1.0 + 0.2 * torch.rand((g, 16, 16, 16), generator=gen, dtype=torch.float64)
    vel = [0.2 * (torch.rand(rho.shape, generator=gen, dtype=torch.float64) - 0.5) for _ in range(3)]
    e = 1.5 + 0.5 * rho * (vel[0] ** 2 + vel[1] ** 2 + vel[2] ** 2)
    u = torch.stack([rho, rho * vel[0], rho * vel[1], rho * vel[2], e], dim=1).float().contiguous().to(dev)
    nbr = torch.arange(g, dtype=torch.int32, device=dev)[:, None].repeat(1, 27).contiguous()      # every group its own neighbour
    out = torch.empty_like(u)
    flux = torch.empty((g, 3, 3, 5, 16, 16), dtype=torch.float32, device=dev)
    gb.gamer_fluid_advance_table_noalloc(u, nbr, out, flux, 1e-3, 1 / 16, G53, gb.MHM, gb.PLM, gb.HLLC)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        gb.gamer_fluid_advance_table_noalloc(u, nbr, out, flux, 1e-3, 1 / 16, G53, gb.MHM, gb.PLM, gb.HLLC)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    assert torch.isfinite(out).all()
    # same options on both sides (n_unphysical_out selects the extended kernel instantiation, whose fp32 multiply-adds the
    # compiler may fuse differently from the fast one's)
    ref = _existing_path(u, nbr, 1e-3, 1 / 16, gb.MHM, gb.PLM, gb.HLLC, {})
    speed, nun = torch.empty_like(ref[2]), torch.zeros(1, dtype=torch.int32, device=dev)
    _noalloc(u, nbr, 1e-3, 1 / 16, gb.MHM, gb.PLM, gb.HLLC, {}, out, flux, speed, nun)
    assert torch.equal(out, ref[0]) and torch.equal(flux, ref[1]) and torch.equal(speed, ref[2])
