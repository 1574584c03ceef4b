"""fp64 CPU oracle of the GAMER-2 patch-group hydro solver -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It never imports paper_1712_07070_b200 (and is never imported by it).
The solver's arithmetic lives in hydro_oracle.c (plain C, gcc) and is only marshalled here; the operations around it are
written out in this file in plain numpy / Python loops: ghost filling (fill_ghosts, fill_ghosts_table), the coarse->fine
ghost interpolation (interpolate_ghosts), the time-step retry loop (fluid_advance_retry) and the SOR Poisson solver
(poisson_sor).  Every function is pinned by tests/test_oracle_*.py; none is "parity unpinned".
"""
import ctypes
import os

import numpy as np

from . import build as _build

MHM, CTU, VL = 1, 2, 3
PLM, PPM = 1, 2
ROE, HLLC, HLLE, EXACT = 1, 2, 3, 4
GMINMOD, VANLEER, VANALBADA = 1, 2, 3

PS, NG, NP = 16, 3, 22


class Opts(ctypes.Structure):
    _fields_ = [
        ("limiter", ctypes.c_int),
        ("theta", ctypes.c_double),
        ("n_scalar", ctypes.c_int),
        ("dual_energy", ctypes.c_int),
        ("de_xi", ctypes.c_double),
        ("min_dens", ctypes.c_double),
        ("min_pres", ctypes.c_double),
        ("min_temp", ctypes.c_double),
        ("remedy_first_order", ctypes.c_int),
        ("char_limiting", ctypes.c_int),
        ("renormalize", ctypes.c_int),
    ]


class Stats(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int64) for n in (
        "n_riemann", "n_riemann_final", "n_roe_fallback", "n_pred_revert",
        "n_first_order", "n_dual_fix", "n_floor", "n_unphysical")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        assert _lib.oracle_sizeof_opts() == ctypes.sizeof(Opts)
        assert _lib.oracle_sizeof_stats() == ctypes.sizeof(Stats)
        _lib.oracle_limited_slope.restype = ctypes.c_double
        _lib.oracle_limited_slope.argtypes = [ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double]
    return _lib


def make_opts(limiter=GMINMOD, theta=0.0, n_scalar=0, dual_energy=False, de_xi=1e-2,
              min_dens=0.0, min_pres=0.0, min_temp=0.0, remedy_first_order=False, char_limiting=False, renormalize=False):
    return Opts(limiter, theta, n_scalar, int(dual_energy), de_xi, min_dens, min_pres, min_temp,
                int(remedy_first_order), int(char_limiting), int(renormalize))


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p) if a is not None else None


def _c64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def set_threads(n):
    os.environ["OMP_NUM_THREADS"] = str(n)


def fluid_advance(u_in, dt, dh, gamma, scheme, recon, riemann, opts=None, want_flux=True):
    """u_in: [G, NV, 22, 22, 22] -> dict(out [G,NV,16,16,16], flux [G,3,3,NV,16,16], speed [G], stats)."""
    u_in = _c64(u_in)
    g, nv = u_in.shape[0], u_in.shape[1]
    assert u_in.shape[2:] == (NP, NP, NP)
    if opts is None:
        opts = make_opts()
    assert nv == 5 + opts.n_scalar
    out = np.empty((g, nv, PS, PS, PS), dtype=np.float64)
    flux = np.empty((g, 3, 3, nv, PS, PS), dtype=np.float64) if want_flux else None
    speed = np.empty((g,), dtype=np.float64)
    st = Stats()
    rc = lib().oracle_fluid_advance(_p(u_in), _p(out), _p(flux), _p(speed), ctypes.c_int64(g),
                                    ctypes.c_double(dt), ctypes.c_double(dh), ctypes.c_double(gamma),
                                    int(scheme), int(recon), int(riemann), ctypes.byref(opts), ctypes.byref(st))
    if rc != 0:
        raise ValueError(f"oracle_fluid_advance returned {rc}")
    return {"out": out, "flux": flux, "speed": speed, "stats": st.as_dict()}


def cfl_dt(u, dh, gamma, cfl, scheme, opts=None):
    """u: [G, NV, 16,16,16] -> (dt, group_speed[G])"""
    u = _c64(u)
    g = u.shape[0]
    if opts is None:
        opts = make_opts(n_scalar=u.shape[1] - 5)
    speed = np.empty((g,), dtype=np.float64)
    dt = ctypes.c_double(0.0)
    rc = lib().oracle_cfl_dt(_p(u), ctypes.c_int64(g), ctypes.c_double(dh), ctypes.c_double(gamma),
                             ctypes.c_double(cfl), int(scheme), ctypes.byref(opts), _p(speed), ctypes.byref(dt))
    if rc != 0:
        raise ValueError(f"oracle_cfl_dt returned {rc}")
    return dt.value, speed


def riemann(solver, axis, UL, UR, gamma, n_scalar=0):
    UL, UR = _c64(UL), _c64(UR)
    F = np.zeros(5 + n_scalar)
    fb = ctypes.c_int(0)
    lib().oracle_riemann(int(solver), int(axis), _p(UL), _p(UR), ctypes.c_double(gamma), int(n_scalar),
                         _p(F), ctypes.byref(fb))
    return F, fb.value


def roe_decomposition(UL, UR, gamma):
    UL, UR = _c64(UL), _c64(UR)
    alpha, lam, K = np.zeros(5), np.zeros(5), np.zeros((5, 5))
    lib().oracle_roe_decomposition(_p(UL), _p(UR), ctypes.c_double(gamma), _p(alpha), _p(lam), _p(K))
    return alpha, lam, K


def limited_slope(limiter, theta, dL, dR):
    return lib().oracle_limited_slope(int(limiter), float(theta), float(dL), float(dR))


def face_values(recon, w5, limiter=GMINMOD, theta=None):
    if theta is None:
        theta = 2.0 if recon == PPM else 1.0
    w5 = _c64(w5)
    wm, wp = ctypes.c_double(0), ctypes.c_double(0)
    lib().oracle_face_values(int(recon), int(limiter), ctypes.c_double(theta), _p(w5),
                             ctypes.byref(wm), ctypes.byref(wp))
    return wm.value, wp.value


def trace_cell(recon, gamma, W, wm, wp, dt_over_dh):
    W, wm, wp = _c64(W), _c64(wm), _c64(wp)
    ns = W.shape[0] - 5
    tm, tp = np.zeros_like(W), np.zeros_like(W)
    lib().oracle_trace_cell(int(recon), ctypes.c_double(gamma), int(ns), _p(W), _p(wm), _p(wp),
                            ctypes.c_double(dt_over_dh), _p(tm), _p(tp))
    return tm, tp


def close_cell(U, gamma, opts):
    U = _c64(U).copy()
    st = Stats()
    ok = lib().oracle_close_cell(_p(U), ctypes.c_double(gamma), ctypes.byref(opts), ctypes.byref(st))
    return U, bool(ok), st.as_dict()


def restrict(fine, coarse, parent):
    """PAPER.md L112 restriction in the group layout: fine [Gf,NV,16,16,16] -> octants of coarse [Gc,NV,16,16,16]
    (modified in place and returned); parent[g] = coarse group * 8 + octant."""
    fine = _c64(fine)
    assert coarse.dtype == np.float64 and coarse.flags["C_CONTIGUOUS"]
    parent = np.ascontiguousarray(parent, dtype=np.int32)
    lib().oracle_restrict(_p(fine), _p(coarse), _p(parent), ctypes.c_int64(fine.shape[0]), int(fine.shape[1]))
    return coarse


def flux_correct(coarse, coarse_flux, fine_flux_avg, table, lam):
    """PAPER.md L112 flux correction of the coarse cells next to coarse-fine boundaries (coarse modified in place);
    table [n, 8] int32 as documented in hydro_oracle.c."""
    assert coarse.dtype == np.float64 and coarse.flags["C_CONTIGUOUS"]
    coarse_flux, fine_flux_avg = _c64(coarse_flux), _c64(fine_flux_avg)
    table = np.ascontiguousarray(table, dtype=np.int32)
    lib().oracle_flux_correct(_p(coarse), _p(coarse_flux), _p(fine_flux_avg), _p(table), ctypes.c_int64(table.shape[0]),
                              int(coarse.shape[1]), ctypes.c_double(lam))
    return coarse


PERIODIC, OUTFLOW, REFLECTING = 0, 1, 2


def fill_ghosts(field, bc=((PERIODIC, PERIODIC),) * 3):
    """Same-level "preparation" step with the standard boundary conditions of L98 on a uniform level:
    field [NV, nz, ny, nx] (conserved; variable 1, 2, 3 = x, y, z momentum) -> padded groups [G, NV, 22, 22, 22],
    g = (gz*Gy + gy)*Gx + gx.  bc = ((x_lo, x_hi), (y_lo, y_hi), (z_lo, z_hi)); a ghost cell c outside [0, n) takes
    the value of cell  c mod n (periodic),  the nearest cell inside (outflow, zero gradient),  or the mirror cell
    -1-c / 2n-1-c with the momentum normal to that face negated (reflecting).  Plain per-axis index tables."""
    field = np.asarray(field)
    nv, nz, ny, nx = field.shape
    n_ax = {0: nx, 1: ny, 2: nz}
    src, flip = {}, {}
    for ax in range(3):
        n = n_ax[ax]
        assert n % PS == 0
        s = np.empty((n // PS, NP), dtype=np.int64)
        f = np.zeros((n // PS, NP), dtype=bool)
        for b in range(n // PS):
            for l in range(NP):
                c = b * PS + l - NG
                if 0 <= c < n:
                    s[b, l] = c
                    continue
                kind = bc[ax][0] if c < 0 else bc[ax][1]
                if kind == PERIODIC:
                    s[b, l] = c % n
                elif kind == OUTFLOW:
                    s[b, l] = 0 if c < 0 else n - 1
                elif kind == REFLECTING:
                    s[b, l] = -1 - c if c < 0 else 2 * n - 1 - c
                    f[b, l] = True
                else:
                    raise ValueError("unknown boundary condition")
        src[ax], flip[ax] = s, f
    gz, gy, gx = nz // PS, ny // PS, nx // PS
    out = np.empty((gz * gy * gx, nv, NP, NP, NP), dtype=field.dtype)
    for bz in range(gz):
        for by in range(gy):
            for bx in range(gx):
                blk = field[:, src[2][bz]][:, :, src[1][by]][:, :, :, src[0][bx]].copy()
                blk[1][:, :, flip[0][bx]] *= -1.0          # x momentum in cells mirrored across an x face
                blk[2][:, flip[1][by], :] *= -1.0
                blk[3][flip[2][bz], :, :] *= -1.0
                out[(bz * gy + by) * gx + bx] = blk
    return out


def char_slope(Wl, Wc, Wr, gamma, limiter=GMINMOD, theta=1.0):
    """Characteristic-limited slope vector of one cell (rotated primitive states of cells j-1, j, j+1)."""
    Wl, Wc, Wr = _c64(Wl), _c64(Wc), _c64(Wr)
    out = np.zeros_like(Wc)
    lib().oracle_char_slope(int(limiter), ctypes.c_double(theta), ctypes.c_double(gamma), int(Wc.shape[0] - 5),
                            _p(Wl), _p(Wc), _p(Wr), _p(out))
    return out


def fill_ghosts_table(u, nbr, padded):
    """Sibling copy of PAPER.md L248 driven by a same-level neighbour table: u [G,NV,16,16,16], nbr [G,27]
    (index (dz+1)*9 + (dy+1)*3 + (dx+1), entry 13 = the group itself, -1 = no same-level neighbour), padded
    [G,NV,22,22,22] modified in place: each of the 27 slabs of a padded group is copied from the group the table names;
    slabs with entry -1 (coarse-fine boundaries, to be interpolated by the caller) are left as they are."""
    u = np.asarray(u)
    rng = {0: (slice(0, NG), slice(PS - NG, PS)), 1: (slice(NG, NG + PS), slice(0, PS)), 2: (slice(NG + PS, NP), slice(0, NG))}
    for g in range(u.shape[0]):
        for dz in range(3):
            for dy in range(3):
                for dx in range(3):
                    s = int(nbr[g, (dz * 3 + dy) * 3 + dx])
                    if s < 0:
                        continue
                    padded[g][:, rng[dz][0], rng[dy][0], rng[dx][0]] = u[s][:, rng[dz][1], rng[dy][1], rng[dx][1]]
    return padded


def fluid_advance_retry(u_in, dt, dh, gamma, scheme, recon, riemann, opts=None, dt_ratio=0.8, dt_min=0.0,
                        want_flux=True):
    """Remedies (iv) and (v) of PAPER.md L107-108 around fluid_advance, in the paper's order: if any cell of the batch
    is still unphysical after the in-solver remedies, "reduce the time-step by a fixed ratio (0.8 by default) and
    recalculate all patches ... with this reduced time-step" (iv); "repeat step (iv) until no unphysical results are
    detected or reaching a given minimum time-step threshold, for which the program is aborted" (v).  The whole batch is
    recomputed from the same u_in each time.  Returns fluid_advance's dict plus "dt_used" and "n_retries"; raises
    FloatingPointError (the abort) when the next reduced step would be below dt_min; after max 200 reductions too.
    Reading (R23): the step of retry k is dt multiplied k times by dt_ratio (not dt * ratio**k), the
    threshold test is dt_k < dt_min, taken before the attempt."""
    n = 0
    while True:
        r = fluid_advance(u_in, dt, dh, gamma, scheme, recon, riemann, opts, want_flux)
        if r["stats"]["n_unphysical"] == 0:
            r["dt_used"], r["n_retries"] = dt, n
            return r
        dt = dt * dt_ratio
        n += 1
        if dt < dt_min or n > 200:
            raise FloatingPointError(f"unphysical cells remain and the reduced time-step {dt} is below dt_min {dt_min}")


def interpolate_ghosts(coarse_padded, parent, nbr, fine_padded, coarse_padded_new=None, w=0.0, monotonic=False):
    """Ghost zones of refined patch groups at coarse-fine boundaries, "interpolating from coarse patches",
    with the "temporal interpolation" between the coarse level's two stored times (L482).  The paper names no spatial
    scheme for the fluid; reading R24: conservative piecewise-linear interpolation of the conserved variables,
        child = U_c + 1/4 * ((+-s_z) + (+-s_y)) + (+-s_x)),  sign + for the upper child along that axis,
    s_d = (U_{c+e_d} - U_{c-e_d}) / 2 (monotonic=False) or minmod(U_c - U_{c-e_d}, U_{c+e_d} - U_c) (monotonic=True), so
    that complete 2x2x2 sets of children average to U_c; U = (1-w) * coarse_padded + w * coarse_padded_new (linear in
    time), or coarse_padded alone when coarse_padded_new is None.
    coarse_padded [Gc,NV,22,22,22] (ghosts already filled); parent[g] = coarse group * 8 + octant (oz*4 + oy*2 + ox) that
    fine group g refines; nbr [Gf,27] the fine level's same-level table: only slabs whose entry is < 0 are written;
    fine_padded [Gf,NV,22,22,22] is modified in place and returned.  Fine cell i (= padded index - 3) along an axis lies
    in coarse cell 8*o + floor(i/2) of the parent group and is its child number i mod 2."""
    cp = np.asarray(coarse_padded, dtype=np.float64)
    if coarse_padded_new is not None:
        cp = (1.0 - w) * cp + w * np.asarray(coarse_padded_new, dtype=np.float64)
    edges = {0: range(0, NG), 1: range(NG, NG + PS), 2: range(NG + PS, NP)}

    def slope(lo, mid, hi):
        if not monotonic:
            return 0.5 * (hi - lo)
        a, b = mid - lo, hi - mid
        return np.where(a * b > 0.0, np.where(np.abs(a) < np.abs(b), a, b), 0.0)

    for g in range(fine_padded.shape[0]):
        cg, o = int(parent[g]) >> 3, int(parent[g]) & 7
        oz, oy, ox = o >> 2, (o >> 1) & 1, o & 1
        C = cp[cg]
        for dz in range(3):
            for dy in range(3):
                for dx in range(3):
                    s = (dz * 3 + dy) * 3 + dx
                    if s == 13 or int(nbr[g, s]) >= 0:
                        continue
                    for pk in edges[dz]:
                        qk, ak = 8 * oz + (pk - NG) // 2 + NG, (pk - NG) % 2
                        for pj in edges[dy]:
                            qj, aj = 8 * oy + (pj - NG) // 2 + NG, (pj - NG) % 2
                            for pi in edges[dx]:
                                qi, ai = 8 * ox + (pi - NG) // 2 + NG, (pi - NG) % 2
                                u = C[:, qk, qj, qi]
                                sz = slope(C[:, qk - 1, qj, qi], u, C[:, qk + 1, qj, qi])
                                sy = slope(C[:, qk, qj - 1, qi], u, C[:, qk, qj + 1, qi])
                                sx = slope(C[:, qk, qj, qi - 1], u, C[:, qk, qj, qi + 1])
                                fine_padded[g, :, pk, pj, pi] = u + 0.25 * (((2 * ak - 1) * sz + (2 * aj - 1) * sy)
                                                                            + (2 * ai - 1) * sx)
    return fine_padded


def poisson_sor(phi, rho, dh, coeff, omega, n_iter, want_acc=True):
    """The refined-level Poisson solver of PAPER.md L126-128 / L236: every patch is relaxed on its own
    (8 + 2*5)^3 = 18^3 grid "with the outermost cells being fixed during the iterations", Laplacian = "its second-order finite
    difference equivalent", method = SOR (Press et al. 2007).  Reading R25: odd-even (red-black) ordering with a
    constant over-relaxation parameter omega and a fixed number of iterations; one iteration = the half-sweep over the
    cells with (i+j+k) even, then the one over the odd cells (i, j, k = indices in the 18^3 array):
        r = phi(i-1) + phi(i+1) + phi(j-1) + phi(j+1) + phi(k-1) + phi(k+1) - 6 phi - coeff dh^2 rho,   phi += omega r / 6
    for  laplacian(phi) = coeff * rho  (coeff = 4 pi G, times the scale factor in comoving coordinates).
    phi [N,18,18,18]: initial guess inside (L238), boundary condition on the outermost layer; rho [N,16,16,16] on the
    relaxed cells.  Returns (phi after n_iter iterations, acc [N,3,8,8,8] or None): acc = -grad(phi) by central
    differences on the 8^3 active zones (cells 5..12 of the 18^3 array, Fig. 2), components ordered (x, y, z)."""
    phi = np.array(phi, dtype=np.float64)
    rho = np.asarray(rho, dtype=np.float64)
    k, j, i = np.meshgrid(np.arange(1, 17), np.arange(1, 17), np.arange(1, 17), indexing="ij")
    src = coeff * dh * dh * rho
    for _ in range(int(n_iter)):
        for colour in (0, 1):
            m = ((k + j + i) % 2 == colour)[None]
            c = phi[:, 1:17, 1:17, 1:17]
            r = (phi[:, 1:17, 1:17, 0:16] + phi[:, 1:17, 1:17, 2:18] + phi[:, 1:17, 0:16, 1:17] + phi[:, 1:17, 2:18, 1:17]
                 + phi[:, 0:16, 1:17, 1:17] + phi[:, 2:18, 1:17, 1:17] - 6.0 * c - src)
            phi[:, 1:17, 1:17, 1:17] = np.where(m, c + omega * r / 6.0, c)
    acc = None
    if want_acc:
        a = slice(5, 13)
        acc = np.stack([-(phi[:, a, a, 6:14] - phi[:, a, a, 4:12]) / (2.0 * dh),
                        -(phi[:, a, 6:14, a] - phi[:, a, 4:12, a]) / (2.0 * dh),
                        -(phi[:, 6:14, a, a] - phi[:, 4:12, a, a]) / (2.0 * dh)], axis=1)
    return phi, acc


def poisson_residual(phi, rho, dh, coeff):
    """Per patch, the largest |phi(i-1) + phi(i+1) + phi(j-1) + phi(j+1) + phi(k-1) + phi(k+1) - 6 phi - coeff dh^2 rho| over
    the 16^3 relaxed cells: dh^2 times the defect of the discretised Poisson equation of PAPER.md L126 (zero "to machine
    precision" once the relaxation has converged).  phi [N,18,18,18], rho [N,16,16,16] -> [N]."""
    phi = np.asarray(phi, dtype=np.float64)
    c = phi[:, 1:17, 1:17, 1:17]
    r = (phi[:, 1:17, 1:17, 0:16] + phi[:, 1:17, 1:17, 2:18] + phi[:, 1:17, 0:16, 1:17] + phi[:, 1:17, 2:18, 1:17]
         + phi[:, 0:16, 1:17, 1:17] + phi[:, 2:18, 1:17, 1:17] - 6.0 * c - coeff * dh * dh * np.asarray(rho, dtype=np.float64))
    return np.abs(r).reshape(phi.shape[0], -1).max(axis=1)


def gravity_update(u, acc, dt):
    """The fluid's gravity update that the paper performs on the GPU "immediately after solving the potential" (
    SURVEY 8(f) NEXT-4 tail; reading R28 of DESIGN.md): with the cell-centred acceleration g = -grad(phi) of a patch's 8^3
    active zones,
        m_new = m + dt * rho * g            (momentum kick; rho is not changed by gravity),
        E_new = E + (|m_new|^2 - |m|^2) / (2 rho)      ("use the corrected momentum to further correct energy", L130:
                                                         the kinetic energy follows the momentum, the thermal energy stays).
    u [G, NV, 16, 16, 16] fluid in the patch-group layout (a copy is returned); acc [8 G, 3, 8, 8, 8] in the PATCH layout
    of poisson_sor, components (x, y, z), patch n = 8 g + octant, octant = oz*4 + oy*2 + ox covering cells
    [8 ox, 8 ox + 8) x [8 oy, ..) x [8 oz, ..) of group g (the octant numbering of restrict / interpolate_ghosts).
    Passive scalars are untouched.  Plain loops over patches; numpy arithmetic inside a patch."""
    u = np.array(u, dtype=np.float64)
    acc = np.asarray(acc, dtype=np.float64)
    assert acc.shape[0] == 8 * u.shape[0] and acc.shape[1:] == (3, 8, 8, 8)
    for n in range(acc.shape[0]):
        g, o = n >> 3, n & 7
        sz, sy, sx = (slice(8 * b, 8 * b + 8) for b in (o >> 2, (o >> 1) & 1, o & 1))
        rho = u[g, 0, sz, sy, sx]
        m_old = [u[g, 1 + d, sz, sy, sx].copy() for d in range(3)]
        m_new = [m_old[d] + (dt * rho) * acc[n, d] for d in range(3)]
        ke_new = (m_new[0] * m_new[0] + m_new[1] * m_new[1]) + m_new[2] * m_new[2]
        ke_old = (m_old[0] * m_old[0] + m_old[1] * m_old[1]) + m_old[2] * m_old[2]
        u[g, 4, sz, sy, sx] = u[g, 4, sz, sy, sx] + 0.5 * (ke_new - ke_old) / rho
        for d in range(3):
            u[g, 1 + d, sz, sy, sx] = m_new[d]
    return u
