"""Two-level AMR harness for BASELINE.json config 3 (test code): a periodic coarse level and one refined
region (ratio 2), one coarse step dt_c and two fine steps dt_c/2, fine ghosts from the coarse
level by conservative linear interpolation in space and linear interpolation in time (L248, L482), then the two
fix-up operations of L112: restriction and flux correction with the solver's `flux_out`.

The solver is a callable (padded [G,NV,22,22,22], dt, dh) -> (out [G,NV,16,16,16], flux [G,3,3,NV,16,16]) so the same
harness drives the CUDA path and the oracle.  Everything here is data movement, interpolation of INPUTS and the
fix-up arithmetic the paper assigns to the AMR driver; none of it is the solver's own arithmetic."""
import torch

from paper_1712_07070_b200 import inputs

PS, NG = 16, 3


def interp_to_fine(cblock):
    """cblock [NV, nz, ny, nx] (with one extra cell per side for the slopes) -> fine [NV, 2(nz-2), 2(ny-2), 2(nx-2)];
    child = parent +- slope/4 per axis with central slopes (conservative: the 8 children average to the parent)."""
    c = cblock[:, 1:-1, 1:-1, 1:-1]
    sz = 0.5 * (cblock[:, 2:, 1:-1, 1:-1] - cblock[:, :-2, 1:-1, 1:-1])
    sy = 0.5 * (cblock[:, 1:-1, 2:, 1:-1] - cblock[:, 1:-1, :-2, 1:-1])
    sx = 0.5 * (cblock[:, 1:-1, 1:-1, 2:] - cblock[:, 1:-1, 1:-1, :-2])
    nv, nz, ny, nx = c.shape
    f = torch.empty((nv, 2 * nz, 2 * ny, 2 * nx), dtype=c.dtype, device=c.device)
    for a in (0, 1):
        for b in (0, 1):
            for d in (0, 1):
                f[:, a::2, b::2, d::2] = c + 0.25 * ((2 * a - 1) * sz + (2 * b - 1) * sy + (2 * d - 1) * sx)
    return f


def pack_fine(uf, uc_t, region):
    """Padded fine batch: interior from uf, ghosts outside the refined region interpolated from the coarse uc_t."""
    z0, z1, y0, y1, x0, x1 = region
    nz, ny, nx = uc_t.shape[1:]
    m = 2 + 1                                   # 2 coarse cells of margin (4 fine >= 3 ghosts) + 1 for the slopes
    iz = torch.arange(z0 - m, z1 + m, device=uc_t.device) % nz
    iy = torch.arange(y0 - m, y1 + m, device=uc_t.device) % ny
    ix = torch.arange(x0 - m, x1 + m, device=uc_t.device) % nx
    cblock = uc_t[:, iz][:, :, iy][:, :, :, ix]
    ext = interp_to_fine(cblock)                # margin of 4 fine cells around the region
    ext[:, 4:-4, 4:-4, 4:-4] = uf
    ext = ext[:, 1:-1, 1:-1, 1:-1]              # keep 3
    w = ext.unfold(1, PS + 2 * NG, PS).unfold(2, PS + 2 * NG, PS).unfold(3, PS + 2 * NG, PS)   # [NV,Gz,Gy,Gx,22,22,22]
    gz, gy, gx = w.shape[1:4]
    return w.permute(1, 2, 3, 0, 4, 5, 6).reshape(gz * gy * gx, uf.shape[0], 22, 22, 22).contiguous(), (gz, gy, gx)


def face_plane(flux, dims, axis, g_index, plane):
    """flux [G,3,3,NV,16,16] -> [NV, n_b, n_a]: the flux through one plane of faces normal to `axis` across the whole
    level (b, a = the two remaining axes, slower first), taken from plane `plane` of the groups at index g_index."""
    gz, gy, gx = dims
    f = flux.reshape(gz, gy, gx, 3, 3, flux.shape[3], PS, PS)
    if axis == 0:
        p = f[:, :, g_index, 0, plane]          # [gz, gy, NV, 16(z), 16(y)]
    elif axis == 1:
        p = f[:, g_index, :, 1, plane]          # [gz, gx, NV, 16(z), 16(x)]
    else:
        p = f[g_index, :, :, 2, plane]          # [gy, gx, NV, 16(y), 16(x)]
    nb, na = p.shape[0], p.shape[1]
    return p.permute(2, 0, 3, 1, 4).reshape(p.shape[2], nb * PS, na * PS)


def avg2x2(p):
    return 0.25 * (p[:, 0::2, 0::2] + p[:, 0::2, 1::2] + p[:, 1::2, 0::2] + p[:, 1::2, 1::2])


def restrict(uf):
    return 0.125 * sum(uf[:, a::2, b::2, d::2] for a in (0, 1) for b in (0, 1) for d in (0, 1))


def two_level_step(solver, uc, uf, region, dh_c, dt_c, fixup=None, pack_fine_fn=None):
    """Returns (uc_new after fix-up, uf_new, records) where records holds every padded batch / output for parity.
    fixup = None: restriction and flux correction are done right here on the global arrays (torch); otherwise
    fixup(uc1, uf, flux_c, [flux_f of each sub-step], region, dt_c / dh_c) -> corrected uc1 (group-layout
    implementations: the oracle's C functions or the CUDA library, see fixup_in_group_layout).
    pack_fine_fn(uf, uc0, uc1, w, region) -> (padded fine batch, fine group dims) replaces the global-array packing of the
    fine level (sibling copy + interpolation from the coarse level at time weight w between uc0 and uc1)."""
    z0, z1, y0, y1, x0, x1 = region
    rec = {}
    cdims = inputs.group_dims(uc)
    pc = inputs.pack_periodic(uc)
    out_c, flux_c = solver(pc, dt_c, dh_c)
    rec["coarse"] = (pc, out_c, flux_c)
    uc1 = inputs.unpack(out_c, *cdims)
    fsum = {}
    fdims = None
    fine_fluxes = []
    for sub in (0, 1):
        w = 0.5 * sub
        if pack_fine_fn is None:
            uc_t = (1.0 - w) * uc + w * uc1                  # linear in time
            pf, fdims = pack_fine(uf, uc_t, region)
        else:
            pf, fdims = pack_fine_fn(uf, uc, uc1, w, region)
        out_f, flux_f = solver(pf, 0.5 * dt_c, 0.5 * dh_c)
        rec["fine%d" % sub] = (pf, out_f, flux_f)
        fine_fluxes.append(flux_f)
        uf = inputs.unpack(out_f, *fdims)
        for axis, n in ((0, fdims[2]), (1, fdims[1]), (2, fdims[0])):
            for side, (gi, pl) in (("lo", (0, 0)), ("hi", (n - 1, 2))):
                p = 0.5 * avg2x2(face_plane(flux_f, fdims, axis, gi, pl))   # time average over the two sub-steps
                fsum[(axis, side)] = fsum.get((axis, side), 0) + p
    if fixup is not None:
        return fixup(uc1, uf, flux_c, fine_fluxes, region, dt_c / dh_c), uf, rec
    # ---- fix-up 1: restriction (L112)
    uc1 = uc1.clone()
    uc1[:, z0:z1, y0:y1, x0:x1] = restrict(uf)
    # ---- fix-up 2: flux correction of the coarse cells next to the coarse-fine interface (L112)
    lam = dt_c / dh_c
    nz, ny, nx = uc.shape[1:]
    lo = {0: x0, 1: y0, 2: z0}
    hi = {0: x1, 1: y1, 2: z1}
    n_ax = {0: nx, 1: ny, 2: nz}
    for axis in (0, 1, 2):
        for side in ("lo", "hi"):
            face = lo[axis] if side == "lo" else hi[axis]
            assert face % 8 == 0, "coarse-fine interfaces must lie on patch faces"
            gi, pl = (face // PS) % (n_ax[axis] // PS), (face % PS) // 8
            fc = face_plane(flux_c, cdims, axis, gi, pl)     # whole coarse level, [NV, n_b, n_a]
            if axis == 0:
                fc = fc[:, z0:z1, y0:y1]
            elif axis == 1:
                fc = fc[:, z0:z1, x0:x1]
            else:
                fc = fc[:, y0:y1, x0:x1]
            d = lam * (fsum[(axis, side)] - fc)
            cell = (face - 1) % n_ax[axis] if side == "lo" else face % n_ax[axis]
            sgn = -1.0 if side == "lo" else 1.0
            if axis == 0:
                uc1[:, z0:z1, y0:y1, cell] += sgn * d
            elif axis == 1:
                uc1[:, z0:z1, cell, x0:x1] += sgn * d
            else:
                uc1[:, cell, y0:y1, x0:x1] += sgn * d
    return uc1, uf, rec


def sedov_two_level(nzc, nyc, nxc, gamma=5.0 / 3.0, device="cpu", e_blast=1.0, p_amb=1e-5):
    """Coarse periodic level nzc x nyc x nxc, central half refined by 2; ambient rho=1, P=p_amb, v=0; energy e_blast
    spread over the central 2x2x2 fine cells (BASELINE.json config 3).  Returns (uc, uf, region, dh_c)."""
    dh_c = 1.0 / nxc
    region = (nzc // 4, 3 * nzc // 4, nyc // 4, 3 * nyc // 4, nxc // 4, 3 * nxc // 4)
    nzf, nyf, nxf = nzc, nyc, nxc               # half the extent at twice the resolution
    one = torch.ones((nzf, nyf, nxf), dtype=torch.float64, device=device)
    pres = p_amb * one.clone()
    dv = (0.5 * dh_c) ** 3
    pres[nzf // 2 - 1:nzf // 2 + 1, nyf // 2 - 1:nyf // 2 + 1, nxf // 2 - 1:nxf // 2 + 1] = (gamma - 1.0) * e_blast / (8 * dv)
    uf = inputs.prim_to_cons(one, 0 * one, 0 * one, 0 * one, pres, gamma)
    onec = torch.ones((nzc, nyc, nxc), dtype=torch.float64, device=device)
    uc = inputs.prim_to_cons(onec, 0 * onec, 0 * onec, 0 * onec, p_amb * onec, gamma)
    z0, z1, y0, y1, x0, x1 = region
    uc[:, z0:z1, y0:y1, x0:x1] = restrict(uf)
    return uc, uf, region, dh_c


def composite_total(uc, uf, region, dh_c):
    z0, z1, y0, y1, x0, x1 = region
    mask = torch.ones(uc.shape[1:], dtype=torch.bool, device=uc.device)
    mask[z0:z1, y0:y1, x0:x1] = False
    return (uc[:, mask].sum(dim=1) * dh_c ** 3 + uf.sum(dim=(1, 2, 3)) * (0.5 * dh_c) ** 3)


# ---------------------------------------------------------------------------------------------------------------
# group-layout description of the same two-level grid, for the fix-up entry points of the library and of the oracle
# ---------------------------------------------------------------------------------------------------------------
def to_groups(field):
    """[NV, nz, ny, nx] -> [G, NV, 16, 16, 16], g = (gz*Gy + gy)*Gx + gx (inverse of inputs.unpack)."""
    nv, nz, ny, nx = field.shape
    w = field.reshape(nv, nz // PS, PS, ny // PS, PS, nx // PS, PS)
    return w.permute(1, 3, 5, 0, 2, 4, 6).reshape(-1, nv, PS, PS, PS).contiguous()


def region_tables(region, cshape):
    """parent [Gf] and coarse-fine face table [n, 8] (int32; layout documented in include/gamer_hydro.h,
    gamer_flux_correct) of a box-shaped refined region of a periodic coarse level."""
    z0, z1, y0, y1, x0, x1 = region
    nz, ny, nx = cshape
    gcy, gcx = ny // PS, nx // PS
    fz, fy, fx = (z1 - z0) // 8, (y1 - y0) // 8, (x1 - x0) // 8          # fine groups per axis

    def cgroup(Z, Y, X):
        return ((Z // PS) * gcy + Y // PS) * gcx + X // PS

    parent, table = [], []
    for a in range(fz):
        for b in range(fy):
            for c in range(fx):
                g = (a * fy + b) * fx + c
                Z, Y, X = z0 + 8 * a, y0 + 8 * b, x0 + 8 * c              # coarse cell at the group's origin
                parent.append(cgroup(Z, Y, X) * 8 + ((Z % PS) // 8) * 4 + ((Y % PS) // 8) * 2 + (X % PS) // 8)
                for d, idx, n_idx, lo, hi, n_ax in ((0, c, fx, x0, x1, nx), (1, b, fy, y0, y1, ny), (2, a, fz, z0, z1, nz)):
                    for side in (0, 1):
                        if idx != (0 if side == 0 else n_idx - 1):
                            continue
                        face = lo if side == 0 else hi                    # coarse face index along d
                        cell = (face - 1) % n_ax if side == 0 else face % n_ax
                        pos_f = [Z, Y, X]
                        pos_c = [Z, Y, X]
                        pos_f[2 - d] = face % n_ax                        # a cell whose lower face is `face`
                        pos_c[2 - d] = cell
                        plane = (face % PS) // 8
                        if d == 0:
                            b0, a0 = Z % PS, Y % PS
                        elif d == 1:
                            b0, a0 = Z % PS, X % PS
                        else:
                            b0, a0 = Y % PS, X % PS
                        table.append([g, d, side, cgroup(*pos_f), plane, (b0 << 8) | a0, cgroup(*pos_c),
                                      ((pos_c[0] % PS) << 16) | ((pos_c[1] % PS) << 8) | (pos_c[2] % PS)])
    return torch.tensor(parent, dtype=torch.int32), torch.tensor(table, dtype=torch.int32).reshape(-1, 8)


def fixup_in_group_layout(restrict_fn, accumulate_fn, correct_fn):
    """Adapter for two_level_step(fixup=...): restrict_fn(fine_groups, coarse_groups, parent) -> coarse_groups;
    accumulate_fn(acc_or_None, flux, weight) -> acc; correct_fn(coarse_groups, coarse_flux, fine_flux_avg, table, lam)
    -> coarse_groups.  All arrays are torch tensors in the solver's group layouts."""
    def fixup(uc1, uf, flux_c, fine_fluxes, region, lam):
        parent, table = region_tables(region, uc1.shape[1:])
        cdims = inputs.group_dims(uc1)
        cg = restrict_fn(to_groups(uf), to_groups(uc1), parent.to(uc1.device))
        acc = None
        for f in fine_fluxes:
            acc = accumulate_fn(acc, f, 1.0 / len(fine_fluxes))
        cg = correct_fn(cg, flux_c, acc, table.to(uc1.device), lam)
        return inputs.unpack(cg, *cdims)
    return fixup


def region_neighbors(region):
    """Same-level neighbour table [Gf, 27] (int32) of the fine groups of a box-shaped refined region: the group at
    offset (dz, dy, dx), or -1 where that offset leaves the region (a coarse-fine boundary)."""
    z0, z1, y0, y1, x0, x1 = region
    fz, fy, fx = (z1 - z0) // 8, (y1 - y0) // 8, (x1 - x0) // 8
    nbr = torch.full((fz * fy * fx, 27), -1, dtype=torch.int32)
    for a in range(fz):
        for b in range(fy):
            for c in range(fx):
                for dz in (-1, 0, 1):
                    for dy in (-1, 0, 1):
                        for dx in (-1, 0, 1):
                            A, B, C = a + dz, b + dy, c + dx
                            if 0 <= A < fz and 0 <= B < fy and 0 <= C < fx:
                                nbr[(a * fy + b) * fx + c, (dz + 1) * 9 + (dy + 1) * 3 + dx + 1] = (A * fy + B) * fx + C
    return nbr
