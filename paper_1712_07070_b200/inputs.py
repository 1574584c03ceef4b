"""Seeded synthetic inputs shaped like the paper's workloads, and the patch-group packing.

This module serves BOTH the CUDA path (tests, bench, smoke) and the oracle's tests.  It holds
no arithmetic of the method itself: it only builds initial conditions (an equation-of-state
conversion from (rho, v, P) to the conserved variables is part of stating an input) and moves
data between a global periodic array and the ghost-padded patch-group batch
(patch group = 2x2x2 patches of 8^3 = 16^3 cells; L300: 3 ghost zones).

Everything is torch, device-agnostic, fp64; callers round to the run precision.  The recipes
 stand in for the paper's own datasets, which are not available:
Blue Waters KH runs (L332-338, reproduced here from the stated initial condition), cluster-merger
and AGORA initial conditions (L354-628, imitated only in character by `disk_field`).
"""
import math

import numpy as np
import torch

PS = 16          # cells per patch-group edge
NG = 3           # ghost zones per side
NP = PS + 2 * NG  # 22


# ----------------------------------------------------------------------------- packing
def group_dims(field):
    nz, ny, nx = field.shape[-3:]
    assert nx % PS == 0 and ny % PS == 0 and nz % PS == 0
    return nz // PS, ny // PS, nx // PS


def _pad_index(n_groups_axis, n_cells, device):
    base = torch.arange(n_groups_axis, device=device)[:, None] * PS
    off = torch.arange(NP, device=device)[None, :] - NG
    return (base + off) % n_cells          # [G_axis, 22], periodic wrap


def pack_periodic(field, dtype=None):
    """[NV, Nz, Ny, Nx] global periodic array -> [G, NV, 22, 22, 22], g = (gz*Gy + gy)*Gx + gx.

    Ghost values are copies of their owners (bit-identical), as the paper's preparation step
    does for same-level neighbours (L248).
    """
    nv = field.shape[0]
    gz, gy, gx = group_dims(field)
    nz, ny, nx = field.shape[-3:]
    dev = field.device
    iz = _pad_index(gz, nz, dev)[:, None, None, :, None, None]
    iy = _pad_index(gy, ny, dev)[None, :, None, None, :, None]
    ix = _pad_index(gx, nx, dev)[None, None, :, None, None, :]
    out = torch.empty((gz * gy * gx, nv, NP, NP, NP), dtype=dtype or field.dtype, device=dev)
    for v in range(nv):
        out[:, v] = field[v][iz, iy, ix].reshape(gz * gy * gx, NP, NP, NP).to(out.dtype)
    return out


def unpack(out, gz, gy, gx):
    """[G, NV, 16,16,16] -> [NV, gz*16, gy*16, gx*16] (inverse of the interior of pack_periodic)."""
    g, nv = out.shape[:2]
    assert g == gz * gy * gx
    t = out.reshape(gz, gy, gx, nv, PS, PS, PS).permute(3, 0, 4, 1, 5, 2, 6)
    return t.reshape(nv, gz * PS, gy * PS, gx * PS).contiguous()


def interior(padded):
    return padded[..., NG:NG + PS, NG:NG + PS, NG:NG + PS]


# ----------------------------------------------------------------------------- helpers
def prim_to_cons(rho, vx, vy, vz, pres, gamma, entropy=False):
    e = pres / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)
    comps = [rho, rho * vx, rho * vy, rho * vz, e]
    if entropy:
        comps.append(pres / rho ** (gamma - 1.0))      # s = P / rho^(gamma-1)
    return torch.stack(comps, dim=0)


def _centres(n, device):
    return (torch.arange(n, device=device, dtype=torch.float64) + 0.5) / n


def _mode_table(seed, n_modes, kmin, kmax, slope):
    rng = np.random.default_rng(seed)
    ks, amps, phases = [], [], []
    while len(ks) < n_modes:
        k = rng.integers(-kmax, kmax + 1, size=3)
        kk = math.sqrt(float((k * k).sum()))
        if kk < kmin or kk > kmax:
            continue
        ks.append(k)
        amps.append(kk ** slope)
        phases.append(rng.uniform(0.0, 2.0 * math.pi))
    amps = np.array(amps)
    amps *= math.sqrt(2.0 / (amps * amps).sum())      # unit variance of the sum
    return np.array(ks), amps, np.array(phases)


def random_field(shape, seed, kmax, device, n_modes=48, kmin=1, slope=-11.0 / 6.0):
    """Unit-variance smooth periodic field: sum of `n_modes` plane waves with integer wave vectors
    (|k| in [kmin,kmax], in units of 2 pi / box), amplitude ~ |k|^slope, random phases."""
    nz, ny, nx = shape
    ks, amps, phases = _mode_table(seed, n_modes, kmin, kmax, slope)
    x, y, z = _centres(nx, device), _centres(ny, device), _centres(nz, device)
    g = torch.zeros(shape, dtype=torch.float64, device=device)
    two_pi = 2.0 * math.pi
    for (kx, ky, kz), a, ph in zip(ks, amps, phases):
        ex = torch.polar(torch.ones_like(x), two_pi * float(kx) * x)
        ey = torch.polar(torch.ones_like(y), two_pi * float(ky) * y)
        ez = torch.polar(torch.ones_like(z), two_pi * float(kz) * z + float(ph))
        g += float(a) * (ez[:, None, None] * ey[None, :, None] * ex[None, None, :]).real
    return g


# ----------------------------------------------------------------------------- workloads
def sod_field(n=64, gamma=1.4, device="cpu", nyz=None):
    """BASELINE.json config 1: Sod tube along x, left (rho,P)=(1,1), right (0.125,0.1), v=0."""
    nyz = nyz or n
    x = _centres(n, device)[None, None, :].expand(nyz, nyz, n)
    left = x < 0.5
    rho = torch.where(left, 1.0, 0.125).to(torch.float64)
    pres = torch.where(left, 1.0, 0.1).to(torch.float64)
    zero = torch.zeros_like(rho)
    return prim_to_cons(rho, zero, zero, zero, pres, gamma)


def turbulence_field(n, seed, kmax=8, gamma=5.0 / 3.0, sigma=1.0, mach=1.0, device="cpu", shape=None,
                     entropy=False):
    """BASELINE.json configs 2 and 4: log-normal density (sigma), Gaussian velocity at rms Mach
    `mach` (against the sound speed of rho=1, P=1), uniform pressure 1."""
    shape = shape or (n, n, n)
    g = random_field(shape, seed, kmax, device)
    rho = torch.exp(sigma * g - 0.5 * sigma * sigma)
    cs0 = math.sqrt(gamma)
    vs = [random_field(shape, seed + 101 * (c + 1), kmax, device) * (mach * cs0 / math.sqrt(3.0))
          for c in range(3)]
    pres = torch.ones_like(rho)
    return prim_to_cons(rho, vs[0], vs[1], vs[2], pres, gamma, entropy=entropy)


def disk_field(nx, ny, nz, seed, gamma=5.0 / 3.0, device="cpu", contrast=1e6, v_rot=20.0, v_jump=100.0,
               n_planes=8):
    """BASELINE.json config 5 (stress): exponential disk, density contrast 1e6 with 10% log-normal
    noise, isothermal T=P/rho=1, flat rotation at v_rot sound speeds, converging velocity jumps of
    v_jump sound speeds across random axis-aligned planes; entropy scalar carried along."""
    x = _centres(nx, device)[None, None, :] - 0.5
    y = _centres(ny, device)[None, :, None] - 0.5
    zext = nz / nx
    z = (_centres(nz, device)[:, None, None] - 0.5) * zext
    r = torch.sqrt(x * x + y * y)
    rd = 1.0 / 8.0
    zd = rd / 10.0
    prof = torch.exp(-r / rd) * torch.exp(-z.abs() / zd)
    prof = torch.clamp(prof, min=1.0 / contrast)
    g = random_field((nz, ny, nx), seed, 8, device)
    rho = prof * torch.exp(0.1 * g)
    cs = math.sqrt(gamma)
    rs = torch.sqrt(r * r + (2.0 / nx) ** 2)
    vx = (-v_rot * cs) * y / rs * torch.ones_like(rho)
    vy = (v_rot * cs) * x / rs * torch.ones_like(rho)
    vz = torch.zeros_like(rho)
    rng = np.random.default_rng(seed + 7)
    coords = [x * torch.ones_like(rho), y * torch.ones_like(rho), z * torch.ones_like(rho)]
    ext = [1.0, 1.0, zext]
    vel = [vx, vy, vz]
    for _ in range(n_planes):
        a = int(rng.integers(0, 3))
        p = float(rng.uniform(-0.4, 0.4)) * ext[a]
        vel[a] = vel[a] - 0.5 * v_jump * cs * torch.sign(coords[a] - p)
    pres = rho.clone()                                   # T = P/rho = 1
    return prim_to_cons(rho, vel[0], vel[1], vel[2], pres, gamma, entropy=True)


def kh_field(n, seed=338, gamma=1.4, device="cpu"):
    """The paper's own uniform-grid workload: shear layers in z, white-noise
    velocity perturbation of amplitude 1e-2."""
    z = _centres(n, device)[:, None, None].expand(n, n, n)
    band = ((z > 0.0) & (z < 0.25)) | ((z > 0.5) & (z < 0.75))
    rho = torch.where(band, 2.0, 1.0).to(torch.float64)
    vx = torch.where(band, 0.5, -0.5).to(torch.float64)
    gen = torch.Generator(device="cpu").manual_seed(seed)
    noise = [(torch.rand((n, n, n), generator=gen, dtype=torch.float64) * 2.0 - 1.0).to(device) * 1e-2
             for _ in range(3)]
    pres = torch.full_like(rho, 2.5)
    return prim_to_cons(rho, vx + noise[0], noise[1], noise[2], pres, gamma)


def blob_field(n, gamma=5.0 / 3.0, device="cpu", v=(1.0, 0.5, -0.75)):
    """Smooth advected density blob at uniform pressure and velocity (stability / symmetry tests)."""
    x = _centres(n, device)[None, None, :]
    y = _centres(n, device)[None, :, None]
    z = _centres(n, device)[:, None, None]
    rho = 1.0 + 0.5 * torch.sin(2 * math.pi * x) * torch.cos(2 * math.pi * y) * torch.cos(4 * math.pi * z)
    one = torch.ones_like(rho)
    return prim_to_cons(rho, v[0] * one, v[1] * one, v[2] * one, one.clone(), gamma)
