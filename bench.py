#!/usr/bin/env python
"""bench.py -- hydro cell-updates/s of the patch-group solver on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--scheme mhm|ctu] [--recon plm|ppm] [--riemann roe|hllc|hlle] [--precision fp32|fp64]
                    [--groups G]

A "step" is one pass of the whole hot path over one batch: gamer_fluid_advance_ex (stage, primitives,
reconstruction, predictor, Riemann, update, boundary fluxes, fused per-group CFL maximum) followed by
gamer_cfl_from_group_speed (dt for the next step).  Default workload = BASELINE.json configs[3]:
32,768 patch groups (512^3 cells) of seeded Mach-1 log-normal turbulence, gamma = 5/3, fp32 MHM+PLM+Roe.
Inputs (7 GB) are far larger than L2 (126 MB), so no L2 flush is needed between iterations.
For N > 1 every rank owns its own 32,768 groups (weak scaling; groups are independent, the only exchange
is the max-reduction of one scalar for dt).

--impl reference times the fp64 CPU oracle (oracle/, test infrastructure) on a bounded sample.
"""
import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

SCHEMES = {"mhm": 1, "ctu": 2, "vl": 3}
RECONS = {"plm": 1, "ppm": 2}
SOLVERS = {"roe": 1, "hllc": 2, "hlle": 3, "exact": 4}
CELLS = 4096

# algorithmic HBM bytes per cell update: padded read + interior write + 9 flux planes
#   PLM needs 5*20^3 values in, PPM 5*22^3; out 5*16^3; flux 9*5*16^2; + 1 speed value per group
def algorithmic_bytes_per_cell(recon, sz, nv=5):
    n_in = nv * (20 ** 3 if recon == 1 else 22 ** 3)
    return (n_in + nv * CELLS + 9 * nv * 256 + 1) * sz / CELLS


# counted SASS FLOPs per cell update (FMA = 2; profiles/flops_per_cell.json from the ncu captures), used for the ALU roofline
FLOPS_PER_CELL = {}


def load_flops():
    p = os.path.join(ROOT, "profiles", "flops_per_cell.json")
    if os.path.exists(p):
        FLOPS_PER_CELL.update(json.load(open(p)))


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d.get("hbm_gbs", 6650.0), d.get("sm_max_mhz", 1965.0), "measured"
    return 6650.0, 1965.0, "fallback"


class ClockSampler(threading.Thread):
    """SM clock and throttle reasons during the timed region (B200_PROFILING.md recipe), sampled through NVML
    (the same counters nvidia-smi prints) every 20 ms."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.stop_flag = index, [], False
        self.max_mhz = None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = int(vis.split(",")[self.index]) if vis and vis.split(",")[self.index].isdigit() else self.index
            h = nv.nvmlDeviceGetHandleByIndex(idx)
            self.max_mhz = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            while not self.stop_flag:
                mhz = nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)
                reasons = nv.nvmlDeviceGetCurrentClocksEventReasons(h) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
                    else nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                self.samples.append((float(mhz), int(reasons)))
                time.sleep(0.01)
        except Exception as e:       # no NVML: report nothing rather than guess
            self.error = repr(e)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        mhz = sorted(s[0] for s in self.samples)
        bits = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20}
        reasons = sorted(n for n, b in bits.items() if any(s[1] & b for s in self.samples))
        return {"sm_mhz": mhz[len(mhz) // 2], "sm_min_mhz": mhz[0], "sm_max_mhz": self.max_mhz, "reasons": reasons,
                "samples": len(mhz)}


def reference_arm(args):
    """The fp64 CPU oracle, as it stands, on a bounded sample of the same workload (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    # torchrun pins OMP_NUM_THREADS=1 for its workers; only this rank works, so it takes all host cores (set before
    # the OpenMP runtime is loaded with torch / the oracle library)
    os.environ["OMP_NUM_THREADS"] = str(os.cpu_count())
    import numpy as np
    import torch
    import oracle
    from paper_1712_07070_b200 import inputs
    scheme, recon, solver = SCHEMES[args.scheme], RECONS[args.recon], SOLVERS[args.riemann]
    n_sample = 512                                                      # 2.1e6 cells, the paper's saturation size
    f = inputs.turbulence_field(128, 7070, kmax=16, gamma=5.0 / 3.0)     # 512 groups of the same field family
    padded = inputs.pack_periodic(f)
    if args.precision == "fp32":
        padded = padded.to(torch.float32).to(torch.float64)
    p = padded.numpy()
    dh = 1.0 / 512
    dt = oracle.cfl_dt(inputs.interior(padded).contiguous().numpy(), dh, 5.0 / 3.0, 0.4, scheme)[0]
    cores = int(os.environ["OMP_NUM_THREADS"])
    for _ in range(max(1, min(args.warmup, 1))):
        oracle.fluid_advance(p, dt, dh, 5.0 / 3.0, scheme, recon, solver)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        r = oracle.fluid_advance(p, dt, dh, 5.0 / 3.0, scheme, recon, solver)
        oracle.cfl_dt(r["out"], dh, 5.0 / 3.0, 0.4, scheme)
    el = time.perf_counter() - t0
    value = n_sample * CELLS * args.steps / el
    sample = f"{n_sample} of 32768 patch groups (128^3 cells of the same field family), {args.steps} steps"
    line = {"impl": "reference", "metric": "hydro cell-updates/sec", "value": value, "unit": "cells/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": el / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(args, n_sample),
            "cpu_baseline": {"value": value, "unit": "cells/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "cells/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def workload_config(args, groups):
    return {"workload": "BASELINE.json configs[3]: seeded Mach-1 log-normal turbulence, gamma=5/3, 16^3 patch groups + 3 ghosts",
            "patch_groups_per_gpu": groups, "cells_per_gpu": groups * CELLS,
            "scheme": args.scheme.upper(), "recon": args.recon.upper(), "riemann": args.riemann.upper(),
            "precision": args.precision, "parallelism": f"dp{args.gpus} (independent patch-group shards)",
            "l2": "inputs (>= 7 GB at full size) exceed the 126 MB L2; no flush needed"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scheme", default="mhm", choices=list(SCHEMES))
    ap.add_argument("--recon", default="plm", choices=list(RECONS))
    ap.add_argument("--riemann", default="roe", choices=list(SOLVERS))
    ap.add_argument("--precision", default="fp32", choices=["fp32", "fp64"])
    ap.add_argument("--groups", type=int, default=32768, help="patch groups per GPU (must be a cube of an integer)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-variants", action="store_true", help="skip the other three configs[3] variants")
    ap.add_argument("--no-extras", action="store_true", help="skip the NEXT-row extras (refresh, fix-up, Poisson)")
    args = ap.parse_args()
    if args.impl == "reference":
        if args.steps > 5:
            args.steps = 5
        return reference_arm(args)

    import torch
    import torch.distributed as dist
    from paper_1712_07070_b200 import binding as gb
    from paper_1712_07070_b200 import inputs

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    gb.lib()                                      # fail loudly if the CUDA library is missing
    load_flops()

    scheme, recon, solver = SCHEMES[args.scheme], RECONS[args.recon], SOLVERS[args.riemann]
    dtype = torch.float32 if args.precision == "fp32" else torch.float64
    sz = 4 if dtype == torch.float32 else 8
    gside = round(args.groups ** (1.0 / 3.0))
    assert gside ** 3 == args.groups, "--groups must be a cube"
    n = gside * PS_CELLS
    gamma, dh, cfl = 5.0 / 3.0, 1.0 / n, (0.4 if scheme == 2 else 0.5)

    # ---- synthetic input, built on the device (seed differs per rank: every rank owns its own box)
    field = inputs.turbulence_field(n, 7070 + rank, kmax=16, gamma=gamma, device=dev)
    u_in = inputs.pack_periodic(field, dtype=dtype)
    if world > 1 or args.no_variants:
        del field
    torch.cuda.empty_cache()
    out, flux, speed = gb.alloc_outputs(u_in)
    dt_dev = torch.zeros(1, dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def time_variant(u, o, fl, sp, sch, rec, sol, c, nsteps, nwarm):
        """nwarm untimed + nsteps timed passes of the hot path (advance + dt) on one resident batch; CUDA events on the
        launching stream: whole loop and each advance launch."""
        gb.gamer_cfl_dt(inputs.interior(u[:64]).contiguous(), dh, gamma, c, sch, None, dt_dev)   # a valid first dt
        o_ = gb.make_opts(stream=stream, dt_dev=dt_dev, group_speed_out=sp)

        def one():
            gb.gamer_fluid_advance_ex(u, o, fl, 1.0, dh, gamma, sch, rec, sol, o_)
            gb.gamer_cfl_from_group_speed(sp, dh, c, dt_dev, stream)
            if world > 1:
                dist.all_reduce(dt_dev, op=dist.ReduceOp.MIN)        # the one exchange: 1 scalar

        for _ in range(nwarm):
            one()
        barrier()
        l0 = gb.gamer_launch_count()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        kev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(nsteps)]
        barrier()
        ev0.record(stream)
        for i in range(nsteps):
            kev[i][0].record(stream)
            gb.gamer_fluid_advance_ex(u, o, fl, 1.0, dh, gamma, sch, rec, sol, o_)
            kev[i][1].record(stream)
            gb.gamer_cfl_from_group_speed(sp, dh, c, dt_dev, stream)
            if world > 1:
                dist.all_reduce(dt_dev, op=dist.ReduceOp.MIN)
        ev1.record(stream)
        barrier()
        nl = gb.gamer_launch_count() - l0
        tot = ev0.elapsed_time(ev1)
        kms = sum(a.elapsed_time(b) for a, b in kev) / nsteps
        t = torch.tensor([tot], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ok = bool(torch.isfinite(o).all().item()) and bool(torch.isfinite(dt_dev).all().item())
        return t.item(), kms, nl, ok, one

    opts = gb.make_opts(stream=stream, dt_dev=dt_dev, group_speed_out=speed)
    sampler = ClockSampler(local)
    sampler.start()
    total_ms, kern_ms, launches, finite, step = time_variant(u_in, out, flux, speed, scheme, recon, solver, cfl,
                                                            args.steps, max(args.warmup, 3))
    sampler.stop_flag = True
    cells = args.groups * CELLS
    value = world * cells * args.steps / (total_ms * 1e-3)

    # ---- extra: the same loop with the device-side periodic ghost refresh included (NEXT-1 row)
    refresh_value = None
    a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if world == 1 and not args.no_extras:
        nref = max(2, min(5, args.steps))
        a0.record(stream)
        for _ in range(nref):
            step()
            gb.gamer_refresh_ghosts_periodic(out, u_in, gside, gside, gside, stream)
        a1.record(stream)
        torch.cuda.synchronize()
        refresh_value = cells * nref / (a0.elapsed_time(a1) * 1e-3)
        finite = finite and bool(torch.isfinite(u_in).all().item())
    # ---- extra: the fused form of the same loop (gamer_fluid_advance_resident: unpadded state + neighbour table,
    # ghost zones gathered inside the solver) -- two unpadded buffers ping-pong, no padded batch is touched
    fused_value = None
    if world == 1 and not args.no_extras:
        nbr = gb.gamer_neighbors_periodic(gside, gside, gside, dev)
        ua, ub = out, torch.empty_like(out)
        nref = max(2, min(5, args.steps))
        for it in range(nref + 1):
            if it == 1:
                a0.record(stream)
            gb.gamer_fluid_advance_resident(ua, nbr, ub, flux, 1.0, dh, gamma, scheme, recon, solver, opts)
            gb.gamer_cfl_from_group_speed(speed, dh, cfl, dt_dev, stream)
            ua, ub = ub, ua
        a1.record(stream)
        torch.cuda.synchronize()
        fused_value = cells * nref / (a0.elapsed_time(a1) * 1e-3)
        finite = finite and bool(torch.isfinite(ua).all().item())
        del ub, nbr

    # ---- extra: the L112 fix-up kernels (NEXT-2) on this batch taken as a fine level: restriction of all groups into
    # groups/8 parent groups, and the time-averaging pass over flux_out; both are pure HBM streams
    fixup = None
    if world == 1 and args.groups >= 64 and not args.no_extras:
        nf = (args.groups // 8) * 8
        parent = torch.arange(nf, dtype=torch.int32, device=dev)          # fine g -> octant g % 8 of coarse g // 8
        coarse = torch.empty((nf // 8,) + tuple(out.shape[1:]), dtype=dtype, device=dev)
        acc = torch.empty_like(flux)
        gb.gamer_restrict(out[:nf], coarse, parent, stream)
        gb.gamer_flux_accumulate(acc, flux, 0.5, True, stream)
        b0, b1, b2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        b0.record(stream)
        for _ in range(5):
            gb.gamer_restrict(out[:nf], coarse, parent, stream)
        b1.record(stream)
        for _ in range(5):
            gb.gamer_flux_accumulate(acc, flux, 0.5, False, stream)
        b2.record(stream)
        torch.cuda.synchronize()
        rb = (out[:nf].numel() + coarse.numel()) * sz
        ab = 3 * flux.numel() * sz
        fixup = {"restrict_GBs": rb * 5 / (b0.elapsed_time(b1) * 1e-3) / 1e9, "restrict_bytes": rb,
                 "flux_accumulate_GBs": ab * 5 / (b1.elapsed_time(b2) * 1e-3) / 1e9, "flux_accumulate_bytes": ab,
                 "hbm_peak_GBs": peaks()[0]}
        # coarse->fine ghost interpolation (gamer_interpolate_ghosts, R24): up to 4096 isolated fine groups (all 26 slabs
        # at a coarse-fine boundary) under the padded batch taken as the coarse level; bytes = ghost cells written +
        # the 14^3 coarse cells each octant's stencil covers, read once
        nfi = min(nf, 4096)
        fine_pad = torch.zeros((nfi,) + tuple(u_in.shape[1:]), dtype=dtype, device=dev)
        nbr_cf = torch.full((nfi, 27), -1, dtype=torch.int32, device=dev)
        nbr_cf[:, 13] = torch.arange(nfi, dtype=torch.int32, device=dev)
        gb.gamer_interpolate_ghosts(u_in, fine_pad, parent[:nfi].contiguous(), nbr_cf, monotonic=True, stream=stream)
        b3, b4 = (torch.cuda.Event(enable_timing=True) for _ in range(2))
        b3.record(stream)
        for _ in range(5):
            gb.gamer_interpolate_ghosts(u_in, fine_pad, parent[:nfi].contiguous(), nbr_cf, monotonic=True, stream=stream)
        b4.record(stream)
        torch.cuda.synchronize()
        ib = nfi * u_in.shape[1] * (22 ** 3 - 16 ** 3 + 14 ** 3) * sz
        fixup["interpolate_ghosts_GBs"] = ib * 5 / (b3.elapsed_time(b4) * 1e-3) / 1e9
        fixup["interpolate_ghosts_bytes"] = ib
        finite = finite and bool(torch.isfinite(fine_pad).all().item())
        del coarse, acc, parent, fine_pad, nbr_cf

    # ---- extra: the paper's other GPU solver (NEXT-4), SOR Poisson on 18^3 per 8^3 patch, 60 red-black iterations (what fp32
    # needs to reach round-off from a random guess); "cells" = the 8^3 active zones, as in the paper's Fig. 5
    poisson = None
    if world == 1 and args.groups >= 64 and not args.no_extras:
        npatch = min(8 * args.groups, 65536)
        gsor = torch.Generator(device=dev).manual_seed(1712)
        phi = torch.randn((npatch, 18, 18, 18), generator=gsor, dtype=dtype, device=dev)
        rho_p = torch.randn((npatch, 16, 16, 16), generator=gsor, dtype=dtype, device=dev) + 2.0
        acc_p = torch.empty((npatch, 3, 8, 8, 8), dtype=dtype, device=dev)
        om, nit = 2.0 / (1.0 + math.sin(math.pi / 17)), 60
        gb.gamer_poisson_sor(phi, rho_p, acc_p, dh, 1.0, om, nit, stream)
        p0, p1 = (torch.cuda.Event(enable_timing=True) for _ in range(2))
        p0.record(stream)
        for _ in range(3):
            gb.gamer_poisson_sor(phi, rho_p, acc_p, dh, 1.0, om, nit, stream)
        p1.record(stream)
        torch.cuda.synchronize()
        tsor = p0.elapsed_time(p1) * 1e-3 / 3
        poisson = {"cells_per_s": npatch * 512 / tsor, "patches": npatch, "n_iter": nit, "ms": tsor * 1e3,
                   "relaxations_per_s": npatch * 4096 * nit / tsor,
                   "hbm_GBs": npatch * (2 * 18 ** 3 + 16 ** 3 + 3 * 512) * sz / tsor / 1e9}
        finite = finite and bool(torch.isfinite(phi).all().item()) and bool(torch.isfinite(acc_p).all().item())
        del phi, rho_p, acc_p
        if dtype == torch.float32:      # the same solve in fp64 (its own shared-memory layout), one timed call
            phi = torch.randn((npatch, 18, 18, 18), generator=gsor, dtype=torch.float64, device=dev)
            rho_p = torch.randn((npatch, 16, 16, 16), generator=gsor, dtype=torch.float64, device=dev) + 2.0
            acc_p = torch.empty((npatch, 3, 8, 8, 8), dtype=torch.float64, device=dev)
            gb.gamer_poisson_sor(phi, rho_p, acc_p, dh, 1.0, om, nit, stream)
            p0.record(stream)
            gb.gamer_poisson_sor(phi, rho_p, acc_p, dh, 1.0, om, nit, stream)
            p1.record(stream)
            torch.cuda.synchronize()
            poisson["fp64_cells_per_s"] = npatch * 512 / (p0.elapsed_time(p1) * 1e-3)
            finite = finite and bool(torch.isfinite(phi).all().item())
            del phi, rho_p, acc_p

    # ---- e2e: host buffers through the C ABI, copies inside the timed region.  gamer_fluid_advance_host_resident ships the
    # UNPADDED state + neighbour table (no ghost bytes cross PCIe) for ALL groups of the workload; the two pinned state
    # buffers ping-pong, so every step uploads the state the previous step downloaded
    e2e = None
    if not args.no_e2e:
        ge = args.groups
        nbr_h = gb.gamer_neighbors_periodic(gside, gside, gside, dev).cpu().pin_memory()
        h_a = torch.empty((ge,) + tuple(out.shape[1:]), dtype=dtype, pin_memory=True)
        h_a.copy_(inputs.interior(u_in))
        h_b = torch.empty_like(h_a).pin_memory()
        h_flux = torch.empty((ge,) + tuple(flux.shape[1:]), dtype=dtype, pin_memory=True)
        h_speed = torch.empty((ge,), dtype=dtype, pin_memory=True)
        dt_host = float(dt_dev.item())
        torch.cuda.synchronize()
        gb.gamer_fluid_advance_host_resident(h_a, nbr_h, h_b, h_flux, h_speed, dt_host, dh, gamma, scheme, recon, solver)   # warm-up: allocations
        ne = 5
        barrier()
        t0 = time.perf_counter()
        for _ in range(ne):
            gb.gamer_fluid_advance_host_resident(h_a, nbr_h, h_b, h_flux, h_speed, dt_host, dh, gamma, scheme, recon, solver)
            dt_host = cfl * dh / float(h_speed.max())
            h_a, h_b = h_b, h_a
        el = time.perf_counter() - t0
        tt = torch.tensor([el], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        finite = finite and bool(torch.isfinite(h_a).all().item())
        e2e = {"value": world * ge * CELLS * ne / tt.item(), "unit": "cells/s",
               "h2d_bytes_per_step": (h_a.numel() + h_speed.numel() * 0) * sz + nbr_h.numel() * 4,
               "d2h_bytes_per_step": (h_b.numel() + h_flux.numel() + h_speed.numel()) * sz,
               "patch_groups_per_step": ge, "steps": ne,
               "api": "gamer_fluid_advance_host_resident (pinned host buffers; unpadded state + neighbour table H2D once per step in "
                      "1024-group chunks, fused-ghost kernels per chunk on 3 streams, out / flux_out / group speeds D2H behind them)"}
        del h_a, h_b, h_flux, h_speed, nbr_h
        gb.gamer_release_scratch()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- measured plain-ALU peaks (gamer_alu_peak: dependent-free streams, same process, same clocks)
    hbm_peak, sm_max, which = peaks()
    alu = {}
    for name, kind in (("ffma", gb.ALU_FFMA), ("dfma", gb.ALU_DFMA), ("fmul_fadd", gb.ALU_FMUL_FADD),
                       ("ffma_fmnmx", gb.ALU_FFMA_FMNMX), ("ffma2", gb.ALU_FFMA2), ("ffma2_fmnmx", gb.ALU_FFMA2_FMNMX),
                       ("ffma_mufu", gb.ALU_FFMA_MUFU), ("ffma2_ffma", gb.ALU_FFMA2_FFMA), ("ffma2_iadd", gb.ALU_FFMA2_IADD)):
        tf, gi = gb.gamer_alu_peak(kind, stream)
        alu[name] = {"tflops": tf, "gwarpinst_per_s": gi}
    alu["issue_slots_gwarpinst_per_s"] = 148 * 4 * sm_max * 1e6 / 1e9
    alu["capture_commit"] = FLOPS_PER_CELL.get("capture_commit")

    def roofline_of(sch_name, rec_name, sol_name, prec, kms):
        szv = 4 if prec == "fp32" else 8
        bpc = algorithmic_bytes_per_cell(RECONS[rec_name], szv)
        key = f"{sch_name}_{rec_name}_{sol_name}_{prec}"
        fpc = FLOPS_PER_CELL.get(key)
        lanes = 128 if szv == 4 else 64
        derived = 148 * lanes * 2 * sm_max * 1e6 / 1e12          # TFLOP/s, DESIGN.md "Rooflines"
        measured = alu["ffma" if szv == 4 else "dfma"]["tflops"]
        hbm_ach = bpc * cells / (kms * 1e-3) / 1e9
        # VL runs in mhm_kernel (its VLS instantiation); CTU is the thread-owned ctu_kernel in fp32, the work-list ctu_wl_kernel in fp64
        r = {"kernel": "ctu_kernel" if (sch_name == "ctu" and szv == 4) else ("ctu_wl_kernel" if sch_name == "ctu" else "mhm_kernel")}
        if fpc:
            ach = fpc * cells / (kms * 1e-3) / 1e12
            r.update({"bound": "alu", "achieved": ach, "peak": measured, "unit": "TFLOP/s", "frac": ach / measured,
                      "flops_per_cell": fpc,
                      "peak_source": f"measured {'FFMA' if szv == 4 else 'DFMA'} stream (gamer_alu_peak), {measured:.2f} TFLOP/s "
                                     f"at {sm_max:.0f} MHz max SM clock; derived 148 SMs x {lanes} lanes x 2 x clock = {derived:.2f}",
                      "peak_derived": derived, "frac_of_derived": ach / derived,
                      "flops_capture_commit": FLOPS_PER_CELL.get("capture_commit")})
        else:
            r.update({"bound": "hbm", "achieved": hbm_ach, "peak": hbm_peak, "unit": "GB/s", "frac": hbm_ach / hbm_peak})
        ipc = FLOPS_PER_CELL.get(key + "_inst_per_cell")
        if ipc:      # instruction-issue view of the same launch: warp instructions per second against 1 / clock / SM sub-partition
            issue_peak = alu["issue_slots_gwarpinst_per_s"]
            issue_ach = ipc / 32.0 * cells / (kms * 1e-3) / 1e9
            r["issue"] = {"achieved": issue_ach, "peak": issue_peak, "unit": "G warp-inst/s", "frac": issue_ach / issue_peak,
                          "warp_inst_x32_per_cell": ipc}
        tr = FLOPS_PER_CELL.get(key + "_dram_bytes_per_cell")
        r["traffic"] = tr * cells if tr else None
        r["hbm"] = {"achieved": hbm_ach, "peak": hbm_peak, "unit": "GB/s", "frac": hbm_ach / hbm_peak,
                    "bytes_per_cell": bpc, "peak_source": which}
        r["kernel_ms"] = kms
        return r

    roofline = roofline_of(args.scheme, args.recon, args.riemann, args.precision, kern_ms)

    # ---- the four variants BASELINE.json configs[3] names, on the same batch (fp64: the same field packed in fp64)
    variants = None
    if world == 1 and not args.no_variants:
        variants = []
        vsteps = max(3, min(10, args.steps))
        bufs = {"fp32": (u_in, out, flux, speed) if sz == 4 else None, "fp64": (u_in, out, flux, speed) if sz == 8 else None}
        for sch_name, rec_name, sol_name, prec in (("mhm", "plm", "roe", "fp32"), ("ctu", "ppm", "hllc", "fp32"),
                                                   ("mhm", "plm", "roe", "fp64"), ("ctu", "ppm", "hllc", "fp64")):
            if (sch_name, rec_name, sol_name, prec) == (args.scheme, args.recon, args.riemann, args.precision):
                v_total, v_kms, v_steps, v_ok = total_ms, kern_ms, args.steps, finite
            else:
                if bufs[prec] is None:
                    for other in list(bufs):      # free the other precision's batch first
                        if other != prec and bufs[other] is not None and bufs[other][0] is not u_in:
                            bufs[other] = None
                    torch.cuda.empty_cache()
                    vt = torch.float32 if prec == "fp32" else torch.float64
                    vu = inputs.pack_periodic(field, dtype=vt)
                    bufs[prec] = (vu,) + gb.alloc_outputs(vu)
                vu, vo, vf, vs = bufs[prec]
                sch = SCHEMES[sch_name]
                v_total, v_kms, _, v_ok, _ = time_variant(vu, vo, vf, vs, sch, RECONS[rec_name], SOLVERS[sol_name],
                                                          0.4 if sch == 2 else 0.5, vsteps, 3)
                v_steps = vsteps
            variants.append({"scheme": sch_name.upper(), "recon": rec_name.upper(), "riemann": sol_name.upper(), "precision": prec,
                             "value": cells * v_steps / (v_total * 1e-3), "unit": "cells/s", "steps": v_steps,
                             "ms_per_step": v_total / v_steps, "kernel_ms": v_kms, "outputs_finite": v_ok,
                             "roofline": roofline_of(sch_name, rec_name, sol_name, prec, v_kms)})
            finite = finite and v_ok
        del bufs
        del field
        torch.cuda.empty_cache()

    cpu = None
    if not args.no_cpu and world == 1:       # the oracle beside it: rank 0 at N = 1 only
        import oracle
        ns = 1024
        sample = u_in[:ns].to(torch.float64).cpu().numpy()
        dtv = float(dt_dev.item())
        oracle.fluid_advance(sample[:64], dtv, dh, gamma, scheme, recon, solver)
        t0 = time.perf_counter()
        reps = 0
        while time.perf_counter() - t0 < 10.0 and reps < 50:
            r = oracle.fluid_advance(sample, dtv, dh, gamma, scheme, recon, solver)
            oracle.cfl_dt(r["out"], dh, gamma, cfl, scheme)
            reps += 1
        el = time.perf_counter() - t0
        cpu = {"value": ns * CELLS * reps / el, "unit": "cells/s", "cores": int(os.environ.get("OMP_NUM_THREADS") or os.cpu_count()),
               "kind": "oracle",
               "sample": f"first {ns} of {args.groups} patch groups, {reps} passes, OpenMP over groups"}

    line = {"metric": "hydro cell-updates/sec", "value": value, "unit": "cells/s", "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if sz == 4 else "f64", "data": "synthetic",
            "config": workload_config(args, args.groups), "clocks": sampler.summary(), "e2e": e2e,
            "gpu_launches": launches, "roofline": roofline, "variants": variants, "alu_peaks": alu, "cpu_baseline": cpu,
            "with_ghost_refresh": refresh_value, "with_fused_ghost_refresh": fused_value, "fixup_kernels": fixup, "poisson_sor": poisson, "outputs_finite": finite,
            "paper_context": "P100-PCIe fp32 ~2e8 cells/s incl. PCIe (PAPER.md L318-320); other hardware, not a target"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


PS_CELLS = 16

if __name__ == "__main__":
    main()
