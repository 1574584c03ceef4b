"""Thin ctypes binding of the C ABI in include/gamer_hydro.h -- argument marshalling only.

Every function has the name of the C entry point it calls; torch tensors provide device memory and
streams, nothing else.  The library is loaded lazily and loading fails loudly: there is no CPU or
PyTorch fallback for any step of the path.
"""
import ctypes
import os

import torch

MHM, CTU, VL = 1, 2, 3
PLM, PPM = 1, 2
ROE, HLLC, HLLE, EXACT = 1, 2, 3, 4
FP32, FP64 = 4, 8
GMINMOD, VANLEER, VANALBADA = 1, 2, 3
BC_PERIODIC, BC_OUTFLOW, BC_REFLECTING = 0, 1, 2
PS, NG, NP = 16, 3, 22

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgamerhydro.so")

EXPORTS = ["gamer_fluid_advance", "gamer_fluid_advance_ex", "gamer_fluid_advance_retry", "gamer_cfl_dt", "gamer_cfl_dt_ex",
           "gamer_cfl_from_group_speed", "gamer_refresh_ghosts_periodic", "gamer_refresh_ghosts", "gamer_refresh_ghosts_table", "gamer_interpolate_ghosts", "gamer_fluid_advance_resident",
           "gamer_neighbors_periodic", "gamer_restrict", "gamer_flux_accumulate", "gamer_flux_correct",
           "gamer_poisson_sor", "gamer_poisson_sor_gravity", "gamer_gravity_update", "gamer_fluid_advance_host", "gamer_fluid_advance_host_resident", "gamer_release_scratch", "gamer_alu_peak", "gamer_fluid_advance_table_noalloc", "gamer_noalloc_max_groups",
           "gamer_launch_count", "gamer_strerror", "gamer_version"]


class gamer_opts(ctypes.Structure):
    _fields_ = [
        ("stream", ctypes.c_void_p),
        ("limiter", ctypes.c_int),
        ("minmod_theta", ctypes.c_double),
        ("n_scalar", ctypes.c_int),
        ("dual_energy", ctypes.c_int),
        ("de_xi", ctypes.c_double),
        ("min_dens", ctypes.c_double),
        ("min_pres", ctypes.c_double),
        ("min_temp", ctypes.c_double),
        ("remedy_first_order", ctypes.c_int),
        ("dt_dev", ctypes.c_void_p),
        ("group_speed_out", ctypes.c_void_p),
        ("n_unphysical_out", ctypes.c_void_p),
        ("diag_out", ctypes.c_void_p),
        ("char_limiting", ctypes.c_int),
        ("renormalize", ctypes.c_int),
    ]


class GamerError(RuntimeError):
    pass


_lib = None


def lib():
    """Load libgamerhydro.so (built in-tree by paper_1712_07070_b200.build).  Raises if missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise GamerError(f"{LIB_PATH} is missing: run `python -m paper_1712_07070_b200.build` "
                             "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        i64, dbl, vp, ci = ctypes.c_int64, ctypes.c_double, ctypes.c_void_p, ctypes.c_int
        adv = [vp, vp, vp, i64, dbl, dbl, dbl, ci, ci, ci, ci]
        L.gamer_fluid_advance.argtypes = adv
        L.gamer_fluid_advance_ex.argtypes = adv + [ctypes.POINTER(gamer_opts)]
        L.gamer_fluid_advance_retry.argtypes = adv + [ctypes.POINTER(gamer_opts), dbl, dbl, ctypes.POINTER(dbl),
                                                      ctypes.POINTER(ctypes.c_int32)]
        cfl = [vp, i64, dbl, dbl, dbl, ci, ci, vp, vp]
        L.gamer_cfl_dt.argtypes = cfl
        L.gamer_cfl_dt_ex.argtypes = cfl + [ctypes.POINTER(gamer_opts)]
        L.gamer_cfl_from_group_speed.argtypes = [vp, i64, dbl, dbl, ci, vp, vp]
        L.gamer_refresh_ghosts_periodic.argtypes = [vp, vp, ci, ci, ci, ci, ci, vp]
        L.gamer_refresh_ghosts.argtypes = [vp, vp, ci, ci, ci, ci, ctypes.POINTER(ci), ci, vp]
        L.gamer_refresh_ghosts_table.argtypes = [vp, vp, vp, i64, ci, ci, vp]
        L.gamer_fluid_advance_resident.argtypes = [vp, vp, vp, vp, i64, dbl, dbl, dbl, ci, ci, ci, ci, ctypes.POINTER(gamer_opts)]
        L.gamer_neighbors_periodic.argtypes = [vp, ci, ci, ci, vp]
        L.gamer_poisson_sor.argtypes = [vp, vp, vp, vp, i64, dbl, dbl, dbl, ci, ci, vp]
        L.gamer_poisson_sor_gravity.argtypes = [vp, vp, vp, vp, vp, ci, dbl, i64, dbl, dbl, dbl, ci, ci, vp]
        L.gamer_gravity_update.argtypes = [vp, vp, i64, ci, dbl, ci, vp]
        L.gamer_interpolate_ghosts.argtypes = [vp, vp, dbl, vp, vp, vp, i64, ci, ci, ci, vp]
        L.gamer_restrict.argtypes = [vp, vp, vp, i64, ci, ci, vp]
        L.gamer_flux_accumulate.argtypes = [vp, vp, dbl, i64, ci, ci, ci, vp]
        L.gamer_flux_correct.argtypes = [vp, vp, vp, vp, i64, ci, dbl, ci, vp]
        L.gamer_fluid_advance_host.argtypes = [vp, vp, vp, vp, i64, dbl, dbl, dbl, ci, ci, ci, ci,
                                               ctypes.POINTER(gamer_opts)]
        L.gamer_fluid_advance_host_resident.argtypes = [vp, vp, vp, vp, vp, i64, dbl, dbl, dbl, ci, ci, ci, ci,
                                                        ctypes.POINTER(gamer_opts)]
        L.gamer_fluid_advance_table_noalloc.argtypes = [vp, vp, vp, vp, i64, dbl, dbl, dbl, ci, ci, ci, ci, ctypes.POINTER(gamer_opts)]
        L.gamer_noalloc_max_groups.argtypes = [ci, ci]
        L.gamer_noalloc_max_groups.restype = ctypes.c_int64
        L.gamer_alu_peak.argtypes = [ci, ctypes.POINTER(dbl), ctypes.POINTER(dbl), vp]
        L.gamer_launch_count.restype = ctypes.c_int64
        L.gamer_strerror.restype = ctypes.c_char_p
        L.gamer_strerror.argtypes = [ci]
        _lib = L
    return _lib


def _check(rc, what):
    if rc != 0:
        raise GamerError(f"{what} failed: {rc} ({lib().gamer_strerror(rc).decode()})")


def _precision(t):
    if t.dtype == torch.float32:
        return FP32
    if t.dtype == torch.float64:
        return FP64
    raise GamerError(f"unsupported dtype {t.dtype}")


def _ptr(t, device_type="cuda"):
    if t is None:
        return None
    if t.device.type != device_type:
        raise GamerError(f"expected a {device_type} tensor, got {t.device}")
    if not t.is_contiguous():
        raise GamerError("tensor must be contiguous")
    return ctypes.c_void_p(t.data_ptr())


def _stream_handle(stream=None):
    s = stream if stream is not None else torch.cuda.current_stream()
    return ctypes.c_void_p(s.cuda_stream)


def make_opts(stream=None, limiter=0, minmod_theta=0.0, n_scalar=0, dual_energy=False, de_xi=0.0, min_dens=0.0,
              min_pres=0.0, min_temp=0.0, remedy_first_order=False, dt_dev=None, group_speed_out=None,
              n_unphysical_out=None, diag_out=None, on_device=True, char_limiting=False, renormalize=False):
    o = gamer_opts()
    o.stream = _stream_handle(stream) if on_device else None
    o.limiter, o.minmod_theta, o.n_scalar = int(limiter), float(minmod_theta), int(n_scalar)
    o.dual_energy, o.de_xi = int(bool(dual_energy)), float(de_xi)
    o.min_dens, o.min_pres, o.min_temp = float(min_dens), float(min_pres), float(min_temp)
    o.remedy_first_order = int(bool(remedy_first_order))
    o.dt_dev = _ptr(dt_dev)
    o.group_speed_out = _ptr(group_speed_out)
    o.n_unphysical_out = _ptr(n_unphysical_out)
    o.diag_out = _ptr(diag_out)
    o.char_limiting = int(bool(char_limiting))
    o.renormalize = int(bool(renormalize))
    # keeps the tensors alive as long as the struct and lets the wrappers check their shapes and dtypes
    o._tensors = {"dt_dev": dt_dev, "group_speed_out": group_speed_out, "n_unphysical_out": n_unphysical_out, "diag_out": diag_out}
    return o


def _check_batch(u, out, flux_out, opts, padded, device_type="cuda"):
    """Cheap shape / dtype / device checks of one advance call (the kernels trust their pointers): u [G,NV,22^3] (padded) or
    [G,NV,16^3], out [G,NV,16,16,16], flux_out [G,3,3,NV,16,16], all of u's dtype; NV = 5 + opts.n_scalar; the optional
    opts outputs: group_speed_out real[G], dt_dev float64[1], n_unphysical_out int32[1], diag_out int32[4] cannot be
    checked from their raw pointers, so make_opts records their tensors."""
    g, nv = int(u.shape[0]), int(u.shape[1])
    edge = NP if padded else PS
    if u.dim() != 5 or tuple(u.shape[2:]) != (edge, edge, edge):
        raise GamerError(f"state must be [G, NV, {edge}, {edge}, {edge}], got {tuple(u.shape)}")
    ns = opts.n_scalar if opts is not None else 0
    if nv != 5 + ns:
        raise GamerError(f"state carries {nv} variables but opts.n_scalar = {ns}")
    if tuple(out.shape) != (g, nv, PS, PS, PS) or out.dtype != u.dtype or out.device.type != device_type:
        raise GamerError(f"out must be [{g}, {nv}, 16, 16, 16] of {u.dtype} on {device_type}")
    if flux_out is not None and (tuple(flux_out.shape) != (g, 3, 3, nv, PS, PS) or flux_out.dtype != u.dtype or flux_out.device.type != device_type):
        raise GamerError(f"flux_out must be [{g}, 3, 3, {nv}, 16, 16] of {u.dtype} on {device_type}")
    for name, shape, dtype in (("group_speed_out", (g,), u.dtype), ("dt_dev", (1,), torch.float64),
                               ("n_unphysical_out", (1,), torch.int32), ("diag_out", (4,), torch.int32)):
        t = getattr(opts, "_tensors", {}).get(name) if opts is not None else None
        if t is not None and (tuple(t.shape) != shape or t.dtype != dtype):
            raise GamerError(f"opts.{name} must be a {dtype} tensor of shape {shape}")


def gamer_fluid_advance(u_in, out, flux_out, dt, dh, gamma, scheme, recon, riemann):
    """11-argument form.  NOTE: runs on the default stream, as the C ABI states."""
    _check_batch(u_in, out, flux_out, None, True)
    n = u_in.shape[0]
    _check(lib().gamer_fluid_advance(_ptr(u_in), _ptr(out), _ptr(flux_out), n, float(dt), float(dh), float(gamma),
                                     int(scheme), int(recon), int(riemann), _precision(u_in)), "gamer_fluid_advance")


def gamer_fluid_advance_ex(u_in, out, flux_out, dt, dh, gamma, scheme, recon, riemann, opts):
    _check_batch(u_in, out, flux_out, opts, True)
    n = u_in.shape[0]
    _check(lib().gamer_fluid_advance_ex(_ptr(u_in), _ptr(out), _ptr(flux_out), n, float(dt), float(dh), float(gamma),
                                        int(scheme), int(recon), int(riemann), _precision(u_in), ctypes.byref(opts)),
           "gamer_fluid_advance_ex")


def gamer_fluid_advance_retry(u_in, out, flux_out, dt, dh, gamma, scheme, recon, riemann, opts, dt_ratio=0.8, dt_min=0.0):
    """Remedies (iv)-(v).  Returns (dt_used, n_retries); GamerError(GAMER_EUNPHYSICAL) = the abort."""
    _check_batch(u_in, out, flux_out, opts, True)
    n = u_in.shape[0]
    dt_used, n_retries = ctypes.c_double(0.0), ctypes.c_int32(0)
    _check(lib().gamer_fluid_advance_retry(_ptr(u_in), _ptr(out), _ptr(flux_out), n, float(dt), float(dh), float(gamma),
                                           int(scheme), int(recon), int(riemann), _precision(u_in), ctypes.byref(opts),
                                           float(dt_ratio), float(dt_min), ctypes.byref(dt_used),
                                           ctypes.byref(n_retries)), "gamer_fluid_advance_retry")
    return dt_used.value, n_retries.value


def gamer_cfl_dt(u, dh, gamma, cfl, scheme, group_speed_out, dt_out, opts=None):
    n = u.shape[0]
    if opts is None:
        opts = make_opts(n_scalar=u.shape[1] - 5)
    _check(lib().gamer_cfl_dt_ex(_ptr(u), n, float(dh), float(gamma), float(cfl), int(scheme), _precision(u),
                                 _ptr(group_speed_out), _ptr(dt_out), ctypes.byref(opts)), "gamer_cfl_dt_ex")


def gamer_cfl_from_group_speed(group_speed, dh, cfl, dt_out, stream=None):
    _check(lib().gamer_cfl_from_group_speed(_ptr(group_speed), group_speed.shape[0], float(dh), float(cfl),
                                            _precision(group_speed), _ptr(dt_out), _stream_handle(stream)),
           "gamer_cfl_from_group_speed")


def gamer_refresh_ghosts_periodic(u, u_in, gz, gy, gx, stream=None):
    _check(lib().gamer_refresh_ghosts_periodic(_ptr(u), _ptr(u_in), gz, gy, gx, u.shape[1], _precision(u),
                                               _stream_handle(stream)), "gamer_refresh_ghosts_periodic")


def gamer_refresh_ghosts(u, u_in, gz, gy, gx, bc, stream=None):
    """bc = (x_lo, x_hi, y_lo, y_hi, z_lo, z_hi) of BC_PERIODIC / BC_OUTFLOW / BC_REFLECTING."""
    arr = (ctypes.c_int * 6)(*[int(b) for b in bc])
    _check(lib().gamer_refresh_ghosts(_ptr(u), _ptr(u_in), gz, gy, gx, u.shape[1], arr, _precision(u),
                                      _stream_handle(stream)), "gamer_refresh_ghosts")


def gamer_refresh_ghosts_table(u, u_in, nbr, stream=None):
    """Sibling copy through a [G, 27] int32 neighbour table; slabs whose entry is -1 are left untouched."""
    if nbr.dtype != torch.int32 or tuple(nbr.shape) != (u.shape[0], 27):
        raise GamerError("nbr must be an int32 tensor of shape [n_groups, 27]")
    _check(lib().gamer_refresh_ghosts_table(_ptr(u), _ptr(u_in), _ptr(nbr), u.shape[0], u.shape[1], _precision(u),
                                            _stream_handle(stream)), "gamer_refresh_ghosts_table")


def gamer_interpolate_ghosts(coarse_in, fine_in, parent, nbr, coarse_in_new=None, w=0.0, monotonic=False, stream=None):
    """Coarse->fine ghost interpolation into the slabs of fine_in whose nbr entry is negative."""
    if parent.dtype != torch.int32 or nbr.dtype != torch.int32 or tuple(nbr.shape) != (fine_in.shape[0], 27):
        raise GamerError("parent / nbr must be int32 tensors of shapes [n_fine] and [n_fine, 27]")
    if coarse_in.dtype != fine_in.dtype or (coarse_in_new is not None and coarse_in_new.shape != coarse_in.shape):
        raise GamerError("coarse and fine batches must share dtype; the two coarse batches must share shape")
    _check(lib().gamer_interpolate_ghosts(_ptr(coarse_in), _ptr(coarse_in_new), float(w), _ptr(fine_in), _ptr(parent),
                                          _ptr(nbr), fine_in.shape[0], fine_in.shape[1], int(bool(monotonic)),
                                          _precision(fine_in), _stream_handle(stream)), "gamer_interpolate_ghosts")


def gamer_fluid_advance_resident(u, nbr, out, flux_out, dt, dh, gamma, scheme, recon, riemann, opts=None):
    """Unpadded state + same-level neighbour table in, unpadded state out: the ghost refresh is fused into the kernel."""
    if nbr.dtype != torch.int32 or tuple(nbr.shape) != (u.shape[0], 27):
        raise GamerError("nbr must be an int32 tensor of shape [n_groups, 27]")
    if opts is None:
        opts = make_opts(n_scalar=u.shape[1] - 5)
    _check_batch(u, out, flux_out, opts, False)
    _check(lib().gamer_fluid_advance_resident(_ptr(u), _ptr(nbr), _ptr(out), _ptr(flux_out), u.shape[0], float(dt), float(dh),
                                              float(gamma), int(scheme), int(recon), int(riemann), _precision(u),
                                              ctypes.byref(opts)), "gamer_fluid_advance_resident")


def gamer_noalloc_max_groups(nvar, precision):
    return int(lib().gamer_noalloc_max_groups(int(nvar), int(precision)))


def gamer_fluid_advance_table_noalloc(u, nbr, out, flux_out, dt, dh, gamma, scheme, recon, riemann, opts=None):
    """Allocation-free step from the unpadded state + neighbour table: the padded batch lives in the library's static
    64 MiB device array (GAMER_ETOOLARGE = -5 beyond gamer_noalloc_max_groups); overlapping calls race on it."""
    if nbr.dtype != torch.int32 or tuple(nbr.shape) != (u.shape[0], 27):
        raise GamerError("nbr must be an int32 tensor of shape [n_groups, 27]")
    if opts is None:
        opts = make_opts(n_scalar=u.shape[1] - 5)
    _check_batch(u, out, flux_out, opts, False)
    _check(lib().gamer_fluid_advance_table_noalloc(_ptr(u), _ptr(nbr), _ptr(out), _ptr(flux_out), u.shape[0], float(dt), float(dh),
                                                   float(gamma), int(scheme), int(recon), int(riemann), _precision(u),
                                                   ctypes.byref(opts)), "gamer_fluid_advance_table_noalloc")


def gamer_neighbors_periodic(gz, gy, gx, device, stream=None):
    """[gz*gy*gx, 27] int32 neighbour table of a periodic box of groups."""
    nbr = torch.empty((gz * gy * gx, 27), dtype=torch.int32, device=device)
    _check(lib().gamer_neighbors_periodic(_ptr(nbr), gz, gy, gx, _stream_handle(stream)), "gamer_neighbors_periodic")
    return nbr


def gamer_restrict(fine, coarse, parent, stream=None):
    """PAPER.md L112 restriction: fine [Gf,NV,16,16,16] into the octants of coarse [Gc,NV,16,16,16] (in place)."""
    if parent.dtype != torch.int32 or parent.shape[0] != fine.shape[0]:
        raise GamerError("parent must be an int32 tensor of length n_fine")
    _check(lib().gamer_restrict(_ptr(fine), _ptr(coarse), _ptr(parent), fine.shape[0], fine.shape[1], _precision(fine),
                                _stream_handle(stream)), "gamer_restrict")


def gamer_flux_accumulate(acc, flux, weight, init, stream=None):
    """acc = (init ? 0 : acc) + weight * flux for flux_out batches [G,3,3,NV,16,16]."""
    _check(lib().gamer_flux_accumulate(_ptr(acc), _ptr(flux), float(weight), flux.shape[0], flux.shape[3], int(bool(init)),
                                       _precision(flux), _stream_handle(stream)), "gamer_flux_accumulate")


def gamer_flux_correct(coarse, coarse_flux, fine_flux_avg, table, lam, stream=None):
    """PAPER.md L112 flux correction of the coarse cells next to coarse-fine boundaries (coarse modified in place)."""
    if table.dtype != torch.int32 or table.dim() != 2 or table.shape[1] != 8:
        raise GamerError("table must be an int32 tensor of shape [n_entries, 8]")
    _check(lib().gamer_flux_correct(_ptr(coarse), _ptr(coarse_flux), _ptr(fine_flux_avg), _ptr(table), table.shape[0],
                                    coarse.shape[1], float(lam), _precision(coarse), _stream_handle(stream)),
           "gamer_flux_correct")


def gamer_poisson_sor(phi, rho, acc, dh, coeff, omega, n_iter, stream=None, resid_out=None):
    """Red-black SOR on every patch's 18^3 potential, in place; acc (nullable) [N,3,8,8,8]."""
    if tuple(phi.shape[1:]) != (18, 18, 18) or tuple(rho.shape) != (phi.shape[0], 16, 16, 16) or rho.dtype != phi.dtype:
        raise GamerError("phi must be [N,18,18,18] and rho [N,16,16,16] of the same dtype")
    if acc is not None and (tuple(acc.shape) != (phi.shape[0], 3, 8, 8, 8) or acc.dtype != phi.dtype):
        raise GamerError("acc must be [N,3,8,8,8] of phi's dtype")
    if resid_out is not None and (tuple(resid_out.shape) != (phi.shape[0],) or resid_out.dtype != phi.dtype):
        raise GamerError("resid_out must be [N] of phi's dtype")
    _check(lib().gamer_poisson_sor(_ptr(phi), _ptr(rho), _ptr(acc), _ptr(resid_out), phi.shape[0], float(dh), float(coeff), float(omega),
                                   int(n_iter), _precision(phi), _stream_handle(stream)), "gamer_poisson_sor")


def _check_gravity(flu, n_patches):
    if flu.dim() != 5 or tuple(flu.shape[2:]) != (PS, PS, PS) or flu.shape[0] * 8 != n_patches:
        raise GamerError("flu must be [n_patches / 8, NV, 16, 16, 16] (patch n = 8 g + octant)")


def gamer_poisson_sor_gravity(phi, rho, acc, flu, dt, dh, coeff, omega, n_iter, stream=None, resid_out=None):
    """gamer_poisson_sor with the fluid's gravity update fused behind the solve; flu in the group layout."""
    if tuple(phi.shape[1:]) != (18, 18, 18) or tuple(rho.shape) != (phi.shape[0], 16, 16, 16) or rho.dtype != phi.dtype or flu.dtype != phi.dtype:
        raise GamerError("phi must be [N,18,18,18], rho [N,16,16,16], flu of the same dtype")
    if acc is not None and (tuple(acc.shape) != (phi.shape[0], 3, 8, 8, 8) or acc.dtype != phi.dtype):
        raise GamerError("acc must be [N,3,8,8,8] of phi's dtype")
    _check_gravity(flu, phi.shape[0])
    _check(lib().gamer_poisson_sor_gravity(_ptr(phi), _ptr(rho), _ptr(acc), _ptr(resid_out), _ptr(flu), flu.shape[1], float(dt),
                                           phi.shape[0], float(dh), float(coeff), float(omega), int(n_iter), _precision(phi),
                                           _stream_handle(stream)), "gamer_poisson_sor_gravity")


def gamer_gravity_update(flu, acc, dt, stream=None):
    """m += dt rho g, E += kinetic-energy difference, for acc [N,3,8,8,8] in the patch layout and flu in the group layout."""
    if tuple(acc.shape[1:]) != (3, 8, 8, 8) or acc.dtype != flu.dtype:
        raise GamerError("acc must be [N,3,8,8,8] of flu's dtype")
    _check_gravity(flu, acc.shape[0])
    _check(lib().gamer_gravity_update(_ptr(flu), _ptr(acc), acc.shape[0], flu.shape[1], float(dt), _precision(flu),
                                      _stream_handle(stream)), "gamer_gravity_update")


def gamer_fluid_advance_host(in_host, out_host, flux_out_host, group_speed_out_host, dt, dh, gamma, scheme, recon,
                             riemann, opts=None):
    """Host-buffer entry: tensors live on the CPU (pinned preferably); copies happen inside the call."""
    n = in_host.shape[0]
    if opts is None:
        opts = make_opts(on_device=False, n_scalar=in_host.shape[1] - 5)
    _check_batch(in_host, out_host, flux_out_host, opts, True, "cpu")
    _check(lib().gamer_fluid_advance_host(_ptr(in_host, "cpu"), _ptr(out_host, "cpu"), _ptr(flux_out_host, "cpu"),
                                          _ptr(group_speed_out_host, "cpu"), n, float(dt), float(dh), float(gamma),
                                          int(scheme), int(recon), int(riemann), _precision(in_host),
                                          ctypes.byref(opts)), "gamer_fluid_advance_host")


def gamer_fluid_advance_host_resident(u_host, nbr_host, out_host, flux_out_host, group_speed_out_host, dt, dh, gamma, scheme,
                                      recon, riemann, opts=None):
    """Host-buffer entry on the UNPADDED state + neighbour table (CPU tensors, pinned preferably); copies happen inside."""
    n = u_host.shape[0]
    if nbr_host.dtype != torch.int32 or tuple(nbr_host.shape) != (n, 27):
        raise GamerError("nbr_host must be an int32 tensor of shape [n_groups, 27]")
    if opts is None:
        opts = make_opts(on_device=False, n_scalar=u_host.shape[1] - 5)
    _check_batch(u_host, out_host, flux_out_host, opts, False, "cpu")
    _check(lib().gamer_fluid_advance_host_resident(_ptr(u_host, "cpu"), _ptr(nbr_host, "cpu"), _ptr(out_host, "cpu"),
                                                   _ptr(flux_out_host, "cpu"), _ptr(group_speed_out_host, "cpu"), n, float(dt),
                                                   float(dh), float(gamma), int(scheme), int(recon), int(riemann),
                                                   _precision(u_host), ctypes.byref(opts)), "gamer_fluid_advance_host_resident")


ALU_FFMA, ALU_FMUL_FADD, ALU_FFMA_FMNMX, ALU_FFMA2, ALU_FFMA2_FMNMX, ALU_DFMA, ALU_FFMA_MUFU, ALU_FFMA2_FFMA, ALU_FFMA2_IADD = range(9)


def gamer_alu_peak(kind, stream=None):
    """Measurement helper: (TFLOP/s, 1e9 warp instructions/s) of a dependent-free instruction stream of the given kind."""
    tf, gi = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(lib().gamer_alu_peak(int(kind), ctypes.byref(tf), ctypes.byref(gi), _stream_handle(stream)), "gamer_alu_peak")
    return tf.value, gi.value


def gamer_release_scratch():
    lib().gamer_release_scratch()


def gamer_launch_count():
    return int(lib().gamer_launch_count())


def gamer_version():
    return int(lib().gamer_version())


# ---------------------------------------------------------------------------------------- allocation helpers
def alloc_outputs(u_in, want_flux=True, want_speed=True):
    """Device buffers of the right shapes for a padded batch [G, NV, 22,22,22]."""
    g, nv = u_in.shape[:2]
    out = torch.empty((g, nv, PS, PS, PS), dtype=u_in.dtype, device=u_in.device)
    flux = torch.empty((g, 3, 3, nv, PS, PS), dtype=u_in.dtype, device=u_in.device) if want_flux else None
    speed = torch.empty((g,), dtype=u_in.dtype, device=u_in.device) if want_speed else None
    return out, flux, speed
