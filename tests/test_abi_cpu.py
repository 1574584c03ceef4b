"""CPU-side checks of the boundary: the C-ABI library loads without a GPU and exports every symbol that
include/gamer_hydro.h declares; the binding mirrors the struct layout.  No compute calls."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built_lib():
    from paper_1712_07070_b200 import build
    return ctypes.CDLL(build.build())


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "gamer_hydro.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gamer_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported(built_lib):
    names = _declared_functions()
    assert "gamer_fluid_advance" in names and "gamer_cfl_dt" in names and len(names) >= 10
    for n in names:
        assert hasattr(built_lib, n), n


def test_binding_lists_the_same_entry_points():
    from paper_1712_07070_b200 import binding
    assert sorted(binding.EXPORTS) == _declared_functions()


def test_version_and_strerror_without_gpu(built_lib):
    built_lib.gamer_strerror.restype = ctypes.c_char_p
    assert built_lib.gamer_version() >= 100
    assert built_lib.gamer_strerror(0) == b"success"
    assert b"invalid" in built_lib.gamer_strerror(-1)


def test_argument_validation_needs_no_gpu(built_lib):
    """Bad arguments are rejected before any CUDA call (error behaviour stated in the header)."""
    L = built_lib
    i64, dbl, vp, ci = ctypes.c_int64, ctypes.c_double, ctypes.c_void_p, ctypes.c_int
    L.gamer_fluid_advance.argtypes = [vp, vp, vp, i64, dbl, dbl, dbl, ci, ci, ci, ci]
    ok = (vp(4096), vp(8192), None)
    assert L.gamer_fluid_advance(None, ok[1], None, 1, 0.1, 0.1, 1.4, 1, 1, 1, 4) == -1
    assert L.gamer_fluid_advance(ok[0], ok[1], None, -1, 0.1, 0.1, 1.4, 1, 1, 1, 4) == -1
    assert L.gamer_fluid_advance(ok[0], ok[1], None, 1, 0.0, 0.1, 1.4, 1, 1, 1, 4) == -1
    assert L.gamer_fluid_advance(ok[0], ok[1], None, 1, float("nan"), 0.1, 1.4, 1, 1, 1, 4) == -1
    assert L.gamer_fluid_advance(ok[0], ok[1], None, 1, 0.1, -1.0, 1.4, 1, 1, 1, 4) == -1
    assert L.gamer_fluid_advance(ok[0], ok[1], None, 1, 0.1, 0.1, 1.0, 1, 1, 1, 4) == -1
    assert L.gamer_fluid_advance(ok[0], ok[1], None, 1, 0.1, 0.1, 1.4, 4, 1, 1, 4) == -1
    assert L.gamer_fluid_advance(ok[0], ok[1], None, 1, 0.1, 0.1, 1.4, 3, 2, 1, 4) == -2      # VL + PPM: fourth ghost zone
    assert L.gamer_fluid_advance(ok[0], ok[1], None, 1, 0.1, 0.1, 1.4, 1, 0, 1, 4) == -1
    assert L.gamer_fluid_advance(ok[0], ok[1], None, 1, 0.1, 0.1, 1.4, 1, 1, 5, 4) == -1
    assert L.gamer_fluid_advance(ok[0], ok[1], None, 1, 0.1, 0.1, 1.4, 1, 1, 1, 2) == -1
    assert L.gamer_fluid_advance(vp(4100), ok[1], None, 1, 0.1, 0.1, 1.4, 1, 1, 1, 4) == -1     # misaligned
    # sizes beyond what the launch grid / 32-bit offsets cover are refused, not truncated
    assert L.gamer_fluid_advance(ok[0], ok[1], None, 1 << 30, 0.1, 0.1, 1.4, 1, 1, 1, 4) == -2
    assert L.gamer_fluid_advance(ok[0], ok[1], None, 0, 0.1, 0.1, 1.4, 1, 1, 1, 4) == 0          # empty batch: no-op
    # extended entry: option fields are validated before any CUDA call
    from paper_1712_07070_b200 import binding as gbo
    L.gamer_fluid_advance_ex.argtypes = [vp, vp, vp, i64, dbl, dbl, dbl, ci, ci, ci, ci, ctypes.POINTER(gbo.gamer_opts)]
    for field, val in (("minmod_theta", 3.0), ("minmod_theta", 0.5), ("n_scalar", 5), ("n_scalar", -1), ("limiter", 9), ("min_dens", -1.0)):
        ob = gbo.gamer_opts()
        setattr(ob, field, val)
        assert L.gamer_fluid_advance_ex(ok[0], ok[1], None, 1, 0.1, 0.1, 1.4, 1, 1, 1, 4, ctypes.byref(ob)) == -1, field
    ob = gbo.gamer_opts()
    ob.dual_energy = 1                                            # needs the entropy scalar
    assert L.gamer_fluid_advance_ex(ok[0], ok[1], None, 1, 0.1, 0.1, 1.4, 1, 1, 1, 4, ctypes.byref(ob)) == -1
    # host entries: the same validation happens before anything is sized or copied; device outputs are refused
    L.gamer_fluid_advance_host.argtypes = [vp, vp, vp, vp, i64, dbl, dbl, dbl, ci, ci, ci, ci, ctypes.POINTER(gbo.gamer_opts)]
    L.gamer_fluid_advance_host_resident.argtypes = [vp, vp, vp, vp, vp, i64, dbl, dbl, dbl, ci, ci, ci, ci, ctypes.POINTER(gbo.gamer_opts)]
    ob = gbo.gamer_opts()
    ob.n_scalar = 7
    assert L.gamer_fluid_advance_host(ok[0], ok[1], None, None, 1, 0.1, 0.1, 1.4, 1, 1, 1, 4, ctypes.byref(ob)) == -1
    assert L.gamer_fluid_advance_host_resident(ok[0], vp(64), ok[1], None, None, 1, 0.1, 0.1, 1.4, 1, 1, 1, 4, ctypes.byref(ob)) == -1
    ob = gbo.gamer_opts()
    ob.diag_out = 4096
    assert L.gamer_fluid_advance_host(ok[0], ok[1], None, None, 1, 0.1, 0.1, 1.4, 1, 1, 1, 4, ctypes.byref(ob)) == -2
    assert L.gamer_fluid_advance_host_resident(None, vp(64), ok[1], None, None, 1, 0.1, 0.1, 1.4, 1, 1, 1, 4, None) == -1
    # fused-refresh entry: no neighbour table, remedy (ii) (needs the padded slab), in-place update
    from paper_1712_07070_b200 import binding as gb
    L.gamer_fluid_advance_resident.argtypes = [vp, vp, vp, vp, i64, dbl, dbl, dbl, ci, ci, ci, ci, ctypes.POINTER(gb.gamer_opts)]
    assert L.gamer_fluid_advance_resident(ok[0], None, ok[1], None, 1, 0.1, 0.1, 1.4, 1, 1, 1, 4, None) == -1
    o = gb.gamer_opts()
    o.remedy_first_order = 1
    assert L.gamer_fluid_advance_resident(ok[0], vp(16384), ok[1], None, 1, 0.1, 0.1, 1.4, 2, 1, 1, 4, ctypes.byref(o)) == -2
    assert L.gamer_fluid_advance_resident(ok[0], vp(16384), ok[0], None, 1, 0.1, 0.1, 1.4, 1, 1, 1, 4, None) == -1
    L.gamer_refresh_ghosts.argtypes = [vp, vp, ci, ci, ci, ci, ctypes.POINTER(ci), ci, vp]
    assert L.gamer_refresh_ghosts(ok[0], ok[1], 1, 1, 1, 5, (ci * 6)(0, 0, 0, 0, 0, 3), 4, None) == -1     # unknown kind
    assert L.gamer_refresh_ghosts(ok[0], ok[1], 1, 1, 1, 5, (ci * 6)(0, 1, 0, 0, 0, 0), 4, None) == -1     # half-periodic axis
    assert L.gamer_refresh_ghosts(ok[0], ok[1], 1, 1, 1, 5, None, 4, None) == -1
    L.gamer_restrict.argtypes = [vp, vp, vp, i64, ci, ci, vp]
    assert L.gamer_restrict(None, ok[1], vp(64), 1, 5, 4, None) == -1
    assert L.gamer_restrict(ok[0], ok[1], vp(64), 1, 10, 4, None) == -1
    assert L.gamer_restrict(ok[0], ok[1], vp(64), 0, 5, 4, None) == 0
    L.gamer_flux_accumulate.argtypes = [vp, vp, dbl, i64, ci, ci, ci, vp]
    assert L.gamer_flux_accumulate(ok[0], None, 0.5, 1, 5, 1, 4, None) == -1
    assert L.gamer_flux_accumulate(ok[0], ok[1], float("inf"), 1, 5, 1, 4, None) == -1
    L.gamer_flux_correct.argtypes = [vp, vp, vp, vp, i64, ci, dbl, ci, vp]
    assert L.gamer_flux_correct(ok[0], ok[1], vp(16384), None, 1, 5, 0.1, 4, None) == -1
    assert L.gamer_flux_correct(ok[0], ok[1], vp(16384), vp(64), 0, 5, 0.1, 4, None) == 0
    L.gamer_neighbors_periodic.argtypes = [vp, ci, ci, ci, vp]
    assert L.gamer_neighbors_periodic(None, 1, 1, 1, None) == -1
    assert L.gamer_neighbors_periodic(vp(4096), 0, 1, 1, None) == -1
    L.gamer_interpolate_ghosts.argtypes = [vp, vp, dbl, vp, vp, vp, i64, ci, ci, ci, vp]
    interp = lambda c0=ok[0], c1=None, w=0.0, f=ok[1], par=vp(64), nb=vp(128), n=1, nv=5, prec=4: \
        L.gamer_interpolate_ghosts(c0, c1, w, f, par, nb, n, nv, 0, prec, None)
    assert interp(c0=None) == -1 and interp(f=None) == -1 and interp(par=None) == -1 and interp(nb=None) == -1
    assert interp(nv=10) == -1 and interp(prec=2) == -1 and interp(n=-1) == -1
    assert interp(c1=vp(16384), w=1.5) == -1 and interp(c1=vp(16384), w=float("nan")) == -1
    assert interp(f=ok[0]) == -1                                # in place
    assert interp(n=0) == 0
    L.gamer_poisson_sor.argtypes = [vp, vp, vp, vp, i64, dbl, dbl, dbl, ci, ci, vp]
    sor = lambda phi=ok[0], rho=ok[1], n=1, dh=0.1, coeff=1.0, omega=1.5, it=10, prec=8: \
        L.gamer_poisson_sor(phi, rho, None, None, n, dh, coeff, omega, it, prec, None)
    assert sor(phi=None) == -1 and sor(rho=None) == -1 and sor(phi=vp(4100)) == -1
    assert sor(omega=2.0) == -1 and sor(omega=0.0) == -1 and sor(dh=0.0) == -1 and sor(it=-1) == -1 and sor(prec=2) == -1
    assert sor(coeff=float("inf")) == -1 and sor(n=-1) == -1
    assert sor(n=0) == 0
    # remedy (iv)/(v) driver: needs opts with the device counter, a host dt, a ratio below 1, dt_min >= 0
    L.gamer_fluid_advance_retry.argtypes = [vp, vp, vp, i64, dbl, dbl, dbl, ci, ci, ci, ci, ctypes.POINTER(gb.gamer_opts),
                                            dbl, dbl, ctypes.POINTER(dbl), ctypes.POINTER(ctypes.c_int32)]
    retry = lambda opts, ratio=0.8, dt_min=0.0, dt=0.1: L.gamer_fluid_advance_retry(
        ok[0], ok[1], None, 1, dt, 0.1, 1.4, 1, 1, 1, 4, opts, ratio, dt_min, None, None)
    assert retry(None) == -1
    o2 = gb.gamer_opts()
    assert retry(ctypes.byref(o2)) == -1                       # no n_unphysical_out
    o2.n_unphysical_out = 32768
    assert retry(ctypes.byref(o2), ratio=1.0) == -1
    assert retry(ctypes.byref(o2), dt_min=-1.0) == -1
    assert retry(ctypes.byref(o2), dt=0.0) == -1
    o2.dt_dev = 65536
    assert retry(ctypes.byref(o2)) == -1                       # dt must live on the host here
    built_lib.gamer_strerror.restype = ctypes.c_char_p
    assert b"unphysical" in built_lib.gamer_strerror(-4)


def test_opts_struct_layout_matches_header():
    from paper_1712_07070_b200 import binding
    fields = [f[0] for f in binding.gamer_opts._fields_]
    text = open(os.path.join(ROOT, "include", "gamer_hydro.h")).read()
    body = text[text.index("typedef struct gamer_opts {"):text.index("} gamer_opts;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    declared = []
    for stmt in body.split("{", 1)[1].split(";"):
        stmt = stmt.strip()
        if not stmt:
            continue
        names = stmt.split(",")
        declared.append(re.findall(r"[A-Za-z_0-9]+", names[0])[-1])
        declared += [re.findall(r"[A-Za-z_0-9]+", n)[-1] for n in names[1:]]
    assert declared == fields


def test_binding_fails_loudly_without_library(monkeypatch, tmp_path):
    from paper_1712_07070_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(binding.GamerError):
        binding.lib()
