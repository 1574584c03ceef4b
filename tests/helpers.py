"""Shared test helpers: oracle-side time loop on a periodic box, error norms."""
import numpy as np
import torch

from paper_1712_07070_b200 import inputs


def load_golden(name):
    import os
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, v = line.split()
            vals[k] = float(v)
    return vals


def oracle_step(oracle, field, dt, dh, gamma, scheme, recon, riemann, opts=None):
    """One step of the oracle on a global periodic field [NV,Nz,Ny,Nx] (torch fp64, cpu)."""
    gz, gy, gx = inputs.group_dims(field)
    padded = inputs.pack_periodic(field)
    r = oracle.fluid_advance(padded.numpy(), dt, dh, gamma, scheme, recon, riemann, opts)
    return inputs.unpack(torch.from_numpy(r["out"]), gz, gy, gx), r


def oracle_run(oracle, field, t_end, dh, gamma, cfl, scheme, recon, riemann, opts=None, max_steps=100000):
    t, n = 0.0, 0
    gz, gy, gx = inputs.group_dims(field)
    while t < t_end * (1 - 1e-12) and n < max_steps:
        u = inputs.pack_periodic(field)
        dt, _ = oracle.cfl_dt(inputs.interior(u).contiguous().numpy(), dh, gamma, cfl, scheme, opts)
        dt = min(dt, t_end - t)
        r = oracle.fluid_advance(u.numpy(), dt, dh, gamma, scheme, recon, riemann, opts, want_flux=False)
        field = inputs.unpack(torch.from_numpy(r["out"]), gz, gy, gx)
        t += dt
        n += 1
    return field, n


def rel_l1(a, b, gamma=None):
    """Relative L1 errors of a conserved batch a against b, [.., NV, ...] with NV on axis 1:
    rho and E (and scalar) per variable; momentum as one vector normalised by sum(|m| + rho c)."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    err = {}
    err["rho"] = np.abs(a[:, 0] - b[:, 0]).sum() / np.abs(b[:, 0]).sum()
    err["E"] = np.abs(a[:, 4] - b[:, 4]).sum() / np.abs(b[:, 4]).sum()
    msum = sum(np.abs(a[:, d] - b[:, d]).sum() for d in (1, 2, 3))
    mabs = np.sqrt(b[:, 1] ** 2 + b[:, 2] ** 2 + b[:, 3] ** 2)
    rho = np.abs(b[:, 0])
    ekin = 0.5 * mabs ** 2 / np.maximum(rho, 1e-300)
    g = gamma if gamma is not None else 5.0 / 3.0
    pres = np.maximum((g - 1.0) * (b[:, 4] - ekin), 0.0)
    rc = np.sqrt(g * pres * rho)
    err["mom"] = msum / (mabs + rc).sum()
    if a.shape[1] > 5:
        err["s"] = np.abs(a[:, 5] - b[:, 5]).sum() / np.abs(b[:, 5]).sum()
    return err
