#!/usr/bin/env python
"""bench.py -- band-H.psi applies per second (complex128) on the 216-atom config (BASELINE.json).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg5] [--impl ours|reference]

A "step" is one full-band apply of the whole hot path: all bands of
the config pushed through qm_apply_h at the config's call batch (cfg5: 512 bands in 32 calls of
16).  Inputs are seeded and synthetic (workloads/), resident in HBM before the timed region.
Prints ONE JSON line (rank 0).  See DESIGN.md section 8 for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "band-H.psi applies/sec (complex128)"
UNIT = "band_applies/s"


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("bf16_tflops", 0.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1590.0, "fallback (B200_PROFILING.md)"


def _ncu_traffic(cfg_name, kernel):
    """DRAM bytes per launch of `kernel` from the committed `ncu --set full` capture (profiles/), or None."""
    p = os.path.join(ROOT, "profiles", f"ncu_traffic_{cfg_name}.json")
    if not os.path.exists(p):
        return None
    return json.load(open(p)).get(kernel)


class ClockSampler(threading.Thread):
    """Samples SM clock / throttle reasons with NVML while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag, self.max_mhz = index, [], set(), False, None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {
                getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
                getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
                getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
                getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            }
            while not self.stop_flag:
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
                time.sleep(0.05)
        except Exception as e:      # no NVML: report it, do not fail the bench
            self.reasons.add(f"nvml_unavailable:{type(e).__name__}")

    def summary(self):
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def _cpu_oracle_rate(cfg, inputs, target_s=12.0):
    """Times the oracle (as it stands) on a bounded sample: one call batch of bands, R sampled output
    rows; cost is affine in R (projections + R rows), so two timings give the full-sphere estimate."""
    from oracle import hpsi as oh
    lat, miller, g2, v, beta, dblk, psi = inputs
    nb = cfg.call_batch
    ng = miller.shape[0]
    vhat = oh.vhat_box(v, cfg.grid)
    d = oh.expand_d(dblk)
    ps = np.ascontiguousarray(psi[:nb])
    rng = np.random.default_rng(7)

    def run(r):
        rows = np.sort(rng.choice(ng, size=min(r, ng), replace=False)).astype(np.int32)
        t = time.perf_counter()
        oh.apply_h_rows(ps, miller, g2, vhat, cfg.grid, beta, d, rows=rows)
        return time.perf_counter() - t, rows.size

    run(16)                 # thread-pool / page warm-up, not used
    t1, r1 = run(64)
    t2, r2 = run(256)
    per_row = max((t2 - t1) / (r2 - r1), 1e-9)
    fixed = max(t1 - per_row * r1, 0.0)
    r3 = int(min(ng, max(256, (target_s - fixed) / per_row)))
    t3, r3 = run(r3)
    per_row = (t3 - fixed) / r3
    t_full = fixed + per_row * ng
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else os.cpu_count()
    omp = os.environ.get("OMP_NUM_THREADS")
    if omp:
        cores = min(cores, int(omp))
    return {"value": nb / t_full, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{cfg.name}: one {nb}-band call batch, {r3} of {ng} sampled output rows "
                      f"({t3:.1f} s measured; projections {fixed:.1f} s + {per_row * 1e3:.2f} ms/row), "
                      f"extrapolated affinely to all rows"}


def _cpu_fft_rate(cfg, inputs, idx):
    """SURVEY 8(d) CPU number (1): the paper's own CPU method -- scatter, library inverse FFT, x V, forward FFT, gather +
    kinetic, projectors as two BLAS products (oracle/hpsi_fft.py) -- on one call batch."""
    from oracle import hpsi as oh
    from oracle import hpsi_fft as of
    lat, miller, g2, v, beta, dblk, psi = inputs
    nb = cfg.call_batch
    d = oh.expand_d(dblk)
    ps = np.ascontiguousarray(psi[:nb])
    of.apply_h_fft(ps[:1], idx, g2, v, cfg.grid, beta, d)            # warm-up (plans, threads)
    t = time.perf_counter()
    of.apply_h_fft(ps, idx, g2, v, cfg.grid, beta, d)
    dt = time.perf_counter() - t
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else os.cpu_count()
    return {"value": nb / dt, "unit": UNIT, "cores": cores, "kind": "oracle-fft (scipy.fft + BLAS zgemm route)",
            "sample": f"{cfg.name}: one {nb}-band call batch, all rows, {dt:.2f} s measured"}


def _build_inputs(cfg, miller_fn):
    from workloads import cell_for, make_beta, make_dmatrix, make_kpoints, make_psi, make_vloc
    lat, pos = cell_for(cfg)
    kpts = make_kpoints(cfg)
    v = make_vloc(cfg, lat)
    dblk = make_dmatrix(cfg)
    per_k = []
    for ik in range(cfg.nk):
        miller = miller_fn(lat, kpts, ik)
        beta = make_beta(cfg, lat, pos, kpts[ik], miller)
        psi = make_psi(cfg, ik, miller.shape[0])
        per_k.append((miller, beta, psi))
    return lat, pos, kpts, v, dblk, per_k


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from workloads import CONFIGS
    from oracle import gsphere as og
    cfg = CONFIGS[args.config]

    def miller_fn(lat, kpts, ik):
        return og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid, kpts[ik])[0]

    lat, pos, kpts, v, dblk, per_k = _build_inputs(cfg, miller_fn)
    miller, idx, g2 = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid, kpts[0])
    inputs = (lat, miller, g2, v, per_k[0][1], dblk, per_k[0][2])
    budget = max(3.0, min(20.0, 150.0 / max(1, args.steps + args.warmup)))
    rates = []
    for s in range(args.warmup + args.steps):
        r = _cpu_oracle_rate(cfg, inputs, target_s=budget)
        if s >= args.warmup:
            rates.append(r)
    val = float(np.mean([r["value"] for r in rates]))
    total_units = cfg.nbands * cfg.nk
    base = dict(rates[-1]); base["value"] = val
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_units / val * 1e3,
            "extrapolated": True,       # each step times a bounded row sample; value / ms_per_step are affine extrapolations
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "complex128",
            "data": "synthetic", "config": _config_dict(cfg, int(idx.size), *_sticks_and_columns(miller, cfg.grid)),
            "cpu_baseline": base,
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def _sticks_and_columns(miller, grid):
    """(z-sticks, x columns) of a sphere from its Miller list: distinct (m1 mod n1, m2 mod n2) pairs and distinct
    m1 mod n1 (the pruned FFT of PAPER.md:733-739 works on these).  Index counting only, no method arithmetic."""
    m = np.asarray(miller, dtype=np.int64)
    a, b = m[:, 0] % grid[0], m[:, 1] % grid[1]
    return int(np.unique(a * grid[1] + b).size), int(np.unique(a).size)


def _config_dict(cfg, ng, nsticks, nx):
    return {"workload": f"{cfg.name}: {cfg.natoms}-atom {'fcc' if cfg.cell == 'fcc' else 'cubic'} Si-like cell, "
                        f"ecutwfc {cfg.ecutwfc_ry:g} Ry, FFT grid {'x'.join(map(str, cfg.grid))}, "
                        f"{cfg.nbands} bands x {cfg.nk} k, {cfg.nproj} projectors, "
                        f"{'dense 4x4 D blocks' if cfg.dense_d else 'diagonal D'}",
            "call_batch": cfg.call_batch, "ng": ng, "sticks": nsticks, "x_columns": nx,
            "cache": "inputs larger than L2 (psi in/out 2x%.0f MB + beta streamed twice per call)" %
                     (cfg.nbands * ng * 16 / 1e6)}


def _verify_timed_output(cfg, lat, kpts, v, dblk, per_k, out_dev, nrows=48):
    """Checks the output of the TIMED steps (last step's psi_out, still on the device) against the direct-sum oracle:
    three bands at the first, a middle and the last call-batch position, `nrows` sampled rows, k-point 0."""
    from oracle import gsphere as og
    from oracle import hpsi as oh
    miller, idx, g2 = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid, kpts[0])
    _, beta, psi = per_k[0]
    ng = idx.size
    nbatch = max(1, cfg.nbands // cfg.call_batch)
    cb = min(cfg.call_batch, cfg.nbands)
    bands = sorted({b * cb + o for b in (0, nbatch // 2, nbatch - 1) for o in (0, cb // 2, cb - 1)})
    rows = np.unique(np.concatenate([[0, ng - 1], np.random.default_rng(17).integers(0, ng, nrows)])).astype(np.int32)
    ref = oh.apply_h_rows(np.ascontiguousarray(psi[bands]), miller, g2, oh.vhat_box(v, cfg.grid), cfg.grid, beta,
                          oh.expand_d(dblk), rows=rows)
    got = out_dev[0][bands][:, rows].cpu().numpy()
    err = float(np.max(np.max(np.abs(got - ref), axis=1) / np.max(np.abs(ref), axis=1)))
    return {"verified": bool(err <= 1e-11), "max_rel_err": err, "bands": [int(b) for b in bands], "rows": int(rows.size),
            "against": "oracle/hpsi_direct.c (direct G-space sum), output of the timed steps"}


def _unfused_figure(qm, torch, dev, hbm_peak):
    """The 512-atom cell (4 x 4 x 4 cubic diamond-structure supercell, a = 41.04 bohr, 30 Ry, 192^3; PAPER.md:1490, 1666 name
    432- and 1024-atom runs): its xy-plane working set exceeds one SM's shared memory, so the library runs the unfused
    y | x | y passes.  Kinetic + local terms of a 16-band batch (the projectors are the same GEMMs as
    everywhere), seeded random psi and V, device-timed; the three slab passes against the HBM roof."""
    lat, ecut, grid, nbb = np.eye(3) * 41.04, 30.0, (192, 192, 192), 16
    gs = qm.GSpace(lat, ecut, grid)
    ng, (nst, nxr) = gs.num_g(0), gs.num_sticks(0)
    gen = torch.Generator(device="cpu")
    gen.manual_seed(512)
    gs.set_vloc(torch.randn(grid, dtype=torch.float64, generator=gen).to(dev))
    gs.set_nonlocal(0, None, None)
    psi = torch.view_as_complex(torch.randn(nbb, ng, 2, dtype=torch.float64, generator=gen)).to(dev)
    out = torch.empty_like(psi)
    for _ in range(3):
        gs.apply_h(psi, out)
    torch.cuda.synchronize()
    qm.qm_profile_enable(gs.handle, True)
    qm.qm_profile_reset(gs.handle)
    reps = 5
    for _ in range(reps):
        gs.apply_h(psi, out)
    torch.cuda.synchronize()
    prof = qm.qm_profile_read(gs.handle)
    qm.qm_profile_enable(gs.handle, False)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        gs.apply_h(psi, out)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    gs.close()
    slab = nbb * nxr * grid[1] * grid[2] * 16            # one copy of the half-transformed planes of the batch
    pass_ms = sum(prof[k][0] for k in ("k_gen_y", "k_gen_x")) / reps
    return {"workload": "512-atom cubic Si-like cell, ecutwfc 30 Ry, FFT grid 192x192x192, kinetic + local terms, "
                        "16-band batch, seeded random psi and V", "ng": ng, "sticks": nst, "x_columns": nxr,
            "ms_per_call": ms, "band_applies_per_s": nbb / (ms * 1e-3),
            "kernel_ms_per_call": {k: v[0] / reps for k, v in prof.items() if v[1]},
            "slab_passes": {"bound": "hbm", "alg_bytes": 4 * slab, "ms": pass_ms, "unit": "GB/s",
                            "achieved": 4 * slab / (pass_ms * 1e-3) / 1e9, "peak": hbm_peak,
                            "frac": 4 * slab / (pass_ms * 1e-3) / 1e9 / hbm_peak,
                            "note": "y backward writes the slab, x reads and writes it, y forward reads it"}}


def _small_config_figure(qm, torch, dev, name, steps, peaks=None, hbm_peak=None):
    """Device-timed applies/s of one of the other BASELINE.json configs (no roofline claim for cfg1-3: launch bound,
    SURVEY 8(d)); same step definition as the headline: all bands x all k at the config's call batch."""
    from workloads import CONFIGS, cell_for, make_kpoints
    cfg = CONFIGS[name]
    lat0, _ = cell_for(cfg)
    gs = qm.GSpace(lat0, cfg.ecutwfc_ry, cfg.grid, make_kpoints(cfg))
    lat, pos, kpts, v, dblk, per_k = _build_inputs(cfg, lambda lat, kpts, ik: gs.miller(ik))
    gs.set_vloc(torch.from_numpy(v).to(dev))
    psi_dev, out_dev = [], []
    for ik, (miller, beta, psi) in enumerate(per_k):
        gs.set_nonlocal(ik, torch.from_numpy(beta).to(dev), torch.from_numpy(dblk).to(dev))
        psi_dev.append(torch.from_numpy(psi).to(dev))
        out_dev.append(torch.empty_like(psi_dev[-1]))
    nb, cb = cfg.nbands, cfg.call_batch
    plan = gs.batch_plan([(ik, psi_dev[ik][b0:b0 + cb], out_dev[ik][b0:b0 + cb])
                          for ik in range(cfg.nk) for b0 in range(0, nb, cb)])

    def step_calls():
        for ik in range(cfg.nk):
            for b0 in range(0, nb, cb):
                gs.apply_h(psi_dev[ik][b0:b0 + cb], out_dev[ik][b0:b0 + cb], k=ik)

    res = {}
    for tag, fn in (("calls", step_calls), ("plan", plan.launch)):
        for _ in range(5):
            fn()
        torch.cuda.synchronize()
        reps = max(steps, 20)
        l0 = gs.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / reps
        res[tag] = (ms, (gs.launch_count() - l0) / reps)
    ver = _verify_timed_output(cfg, lat, kpts, v, dblk, per_k, out_dev, nrows=32)
    ng = gs.num_g(0)
    # per-kernel device time of one step of plain calls (events around every launch; the side stream is off meanwhile)
    qm.qm_profile_enable(gs.handle, True)
    qm.qm_profile_reset(gs.handle)
    step_calls()
    torch.cuda.synchronize()
    prof = qm.qm_profile_read(gs.handle)
    qm.qm_profile_enable(gs.handle, False)
    kern = {k: {"avg_ms": t / n, "launches_per_step": n} for k, (t, n) in prof.items() if n}
    if peaks is not None and "k_plane" in kern:
        # the same two roofs as the headline's plane kernel, per launch of `cb` bands
        dmma_peak, smem_peak = peaks
        n1, n3 = cfg.grid[0], cfg.grid[2]
        nxr = gs.num_sticks(0)[1]
        t = kern["k_plane"]["avg_ms"] * 1e-3
        fl = cb * n3 * ((2 * nxr + 2 * n1) * 5.0 * n1 * np.log2(n1) + 2.0 * n1 * cfg.grid[1])
        by = cb * n3 * (8.0 * n1 * nxr + 4.0 * n1 * n1) * 16.0
        kern["k_plane"].update(bound="alu", achieved=fl / t / 1e12, peak=dmma_peak, unit="TFLOP/s", frac=fl / t / 1e12 / dmma_peak,
                               co_bound={"bound": "smem", "achieved": by / t / 1e12, "peak": smem_peak, "unit": "TB/s",
                                         "frac": by / t / 1e12 / smem_peak})
        # the other kernels of an apply, same work models as the headline's `kernels` (per launch of `cb` bands)
        nst = gs.num_sticks(0)[0]
        for kname, work in (("k_proj1", 6.0 * cfg.nproj * cb * ng), ("k_proj2", 6.0 * cfg.nproj * cb * ng)):
            if kname in kern:
                a = work / (kern[kname]["avg_ms"] * 1e-3) / 1e12
                kern[kname].update(bound="tensor", achieved=a, peak=dmma_peak, unit="TFLOP/s", frac=a / dmma_peak)
        if hbm_peak:
            for kname, work in (("k_zinv", cb * (ng * 16 + n3 * nst * 16)), ("k_zfwd", cb * (n3 * nst * 16 + 2 * ng * 16) + ng * 8)):
                if kname in kern:
                    a = work / (kern[kname]["avg_ms"] * 1e-3) / 1e9
                    kern[kname].update(bound="l2+hbm", achieved=a, peak=hbm_peak, unit="GB/s", frac=a / hbm_peak, alg_bytes=work)
    plan.close()
    gs.close()
    best = min(res, key=lambda t: res[t][0])
    ms = res[best][0]
    ncalls = cfg.nk * ((nb + cb - 1) // cb)
    return {"workload": _config_dict(cfg, ng, 0, 0)["workload"], "call_batch": cb, "band_applies_per_s": nb * cfg.nk / (ms * 1e-3),
            "ms_per_full_band_apply": ms, "us_per_call": ms * 1e3 / ncalls, "calls_per_step": ncalls,
            "launch_mode": best, "ms_by_mode": {t: r[0] for t, r in res.items()},
            "launches_per_call": res["calls"][1] / ncalls, "kernels": kern,
            "verified": ver["verified"], "max_rel_err": ver["max_rel_err"]}


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2308_07277_b200 as qm
    from workloads import CONFIGS

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and there is no CPU fallback (use --impl reference)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    cfg = CONFIGS[args.config]
    hbm_peak, _bf16, peak_src = _peaks()

    from workloads import cell_for, make_kpoints
    lat0, _ = cell_for(cfg)
    gs = qm.GSpace(lat0, cfg.ecutwfc_ry, cfg.grid, make_kpoints(cfg))

    def miller_fn(lat, kpts, ik):
        return gs.miller(ik)

    lat, pos, kpts, v, dblk, per_k = _build_inputs(cfg, miller_fn)
    gs.set_vloc(torch.from_numpy(v).to(dev))
    psi_dev, out_dev = [], []
    for ik, (miller, beta, psi) in enumerate(per_k):
        gs.set_nonlocal(ik, torch.from_numpy(beta).to(dev), torch.from_numpy(dblk).to(dev))
        psi_dev.append(torch.from_numpy(psi).to(dev))
        out_dev.append(torch.empty_like(psi_dev[-1]))
    torch.cuda.synchronize()
    nb, cb = cfg.nbands, cfg.call_batch
    ng = gs.num_g(0)
    nsticks, nx = gs.num_sticks(0)
    assert (nsticks, nx) == _sticks_and_columns(gs.miller(0), cfg.grid)       # what the reference arm prints in `config`

    def step():
        for ik in range(cfg.nk):
            for b0 in range(0, nb, cb):
                gs.apply_h(psi_dev[ik][b0:b0 + cb], out_dev[ik][b0:b0 + cb], k=ik)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(3, args.warmup)):
        step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = gs.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = gs.launch_count() - l0
    verify = None
    if rank == 0 and not args.no_cpu_baseline:
        verify = _verify_timed_output(cfg, lat, kpts, v, dblk, per_k, out_dev)      # output of the timed steps

    # second, instrumented pass of the same steps: per-kernel device time (CUDA events on the launch stream)
    qm.qm_profile_reset(gs.handle)
    qm.qm_profile_enable(gs.handle, True)
    for _ in range(args.steps):
        step()
    torch.cuda.synchronize()
    prof = qm.qm_profile_read(gs.handle)
    qm.qm_profile_enable(gs.handle, False)

    # SURVEY A17 second figure: one qm_apply_h call with all bands of the config (the library runs the FFT path in
    # L2-sized band chunks and the projector GEMMs over the whole block)
    gs.apply_h(psi_dev[0], out_dev[0], k=0)
    torch.cuda.synchronize()
    a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a0.record()
    gs.apply_h(psi_dev[0], out_dev[0], k=0)
    a1.record()
    torch.cuda.synchronize()
    one_call_ms = a0.elapsed_time(a1)

    # next row of the scope table: subspace products <psi_i|H psi_j>, all bands x all bands and one
    # call batch x one call batch, device-timed outside the step timing above (own figure, not part of `value`)
    sub = {}
    for tag, n_sub in (("all_bands", nb), ("call_batch", cb)):
        a_sub, b_sub = psi_dev[0][:n_sub], out_dev[0][:n_sub]
        s_sub = gs.subspace(a_sub, b_sub)
        torch.cuda.synchronize()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 3
        s0.record()
        for _ in range(reps):
            gs.subspace(a_sub, b_sub, s_sub)
        s1.record()
        torch.cuda.synchronize()
        sub[tag] = (n_sub, s0.elapsed_time(s1) / reps)

    # 8(f) rank 2: density accumulation n(r) += f_i |psi_i(r)|^2, one call batch of bands per call, all bands of the config
    occ_dev = torch.full((nb,), 2.0, dtype=torch.float64, device=dev)
    rho_dev = torch.empty(int(np.prod(cfg.grid)), dtype=torch.float64, device=dev)

    def density_pass():
        gs.density_reset()
        for b0 in range(0, nb, cb):
            gs.density_accumulate(psi_dev[0][b0:b0 + cb], occ_dev[b0:b0 + cb])
        gs.density_get(rho_dev)

    density_pass()
    torch.cuda.synchronize()
    d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    d0.record()
    density_pass()
    d1.record()
    torch.cuda.synchronize()
    density_ms = d0.elapsed_time(d1)

    # 8(f) rank 3: Taylor propagator of order 4 (eq. 52) over all bands, one call batch per call
    def taylor_pass():
        for b0 in range(0, nb, cb):
            gs.taylor_propagate(psi_dev[0][b0:b0 + cb], 0.02, 4, out_dev[0][b0:b0 + cb])

    taylor_pass()
    torch.cuda.synchronize()
    y0, y1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    y0.record()
    taylor_pass()
    y1.record()
    torch.cuda.synchronize()
    taylor_ms = y0.elapsed_time(y1)

    # 8(f) rank 3, second half: split-operator step (eq. 53), one call batch per call
    gs.split_operator_set(torch.from_numpy(v).to(dev), 0.02)

    def splitop_pass():
        for b0 in range(0, nb, cb):
            gs.split_operator_propagate(psi_dev[0][b0:b0 + cb], out_dev[0][b0:b0 + cb])

    splitop_pass()
    torch.cuda.synchronize()
    o0, o1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    o0.record()
    splitop_pass()
    o1.record()
    torch.cuda.synchronize()
    splitop_ms = o0.elapsed_time(o1)

    # 8(f) rank 4: GW plane-wave matrix elements (eqs. 56-57), q = 0, 16 x 16 states, epsilon cut-off 10 Ry
    n_me = min(16, nb)
    me = gs.mtxel(0, 0, 10.0)
    me_out = me.apply(psi_dev[0][:n_me], psi_dev[0][nb - n_me:])
    torch.cuda.synchronize()
    m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    m0.record()
    me.apply(psi_dev[0][:n_me], psi_dev[0][nb - n_me:], me_out)
    m1.record()
    torch.cuda.synchronize()
    mtxel_ms = m0.elapsed_time(m1)
    mtxel_ng = me.num_g()
    me.close()
    del me_out

    # end to end through the host entry: pinned host buffers, copies inside the timed region
    hin = [p.cpu().pin_memory() for p in psi_dev]
    hout = [torch.empty_like(h).pin_memory() for h in hin]

    def step_host():
        for ik in range(cfg.nk):
            for b0 in range(0, nb, cb):
                gs.apply_h_host_async(hin[ik][b0:b0 + cb], hout[ik][b0:b0 + cb], k=ik)
        gs.host_synchronize()       # every band's result is back in host memory before the step ends

    step_host()
    step_host()             # two warm-up passes: the host pipeline has two staging slots, each grown on first use
    barrier()
    t0 = time.perf_counter()
    h0, h1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    h0.record()
    e2e_steps = max(1, args.steps)                   # the same number of steps as the device-timed value
    for _ in range(e2e_steps):
        step_host()
    h1.record()
    barrier()
    ms_host = max(h0.elapsed_time(h1), (time.perf_counter() - t0) * 1e3)
    sampler.stop_flag = True
    sampler.join(timeout=2)

    from paper_2308_07277_b200 import dist_util as du
    ms, ms_host = du.max_over_ranks([ms, ms_host], device=dev)
    units_per_step = du.units_per_step(nb * cfg.nk, world, "weak")   # every rank applies H to its own band set
    value = units_per_step * args.steps / (ms * 1e-3)
    e2e_value = units_per_step * e2e_steps / (ms_host * 1e-3)
    bytes_io = nb * cfg.nk * ng * 16

    if rank == 0:
        dmma_peak, dfma_peak = qm.qm_probe_fp64_tensor_peak()
        nproj = cfg.nproj
        S, N3 = nsticks, cfg.grid[2]
        nvox = int(np.prod(cfg.grid))
        # algorithmic work per launch (one call batch `cb` bands), DESIGN.md section 7
        alg = {
            "k_zinv": ("hbm", cb * (ng * 16 + N3 * S * 16)),
            "k_plane": ("alu", cb * N3 * ((2 * nx + 2 * cfg.grid[0]) * 5.0 * cfg.grid[0] * np.log2(cfg.grid[0])
                                          + 2.0 * cfg.grid[0] * cfg.grid[1])),
            "k_zfwd": ("hbm", cb * (N3 * S * 16 + 2 * ng * 16) + ng * 8),
            # executed flops: the 3M scheme issues 3 real DMMA products = 6 flop per complex MAC; `frac` is pipe
            # utilisation (executed / peak).  The textbook 8 flop per complex MAC is reported as `effective_tflops`.
            "k_proj1": ("tensor", 6.0 * nproj * cb * ng),
            "k_proj2": ("tensor", 6.0 * nproj * cb * ng),
        }
        effective = {"k_proj1": 8.0 * nproj * cb * ng, "k_proj2": 8.0 * nproj * cb * ng}
        total_k = sum(v[0] for v in prof.values()) or 1.0
        kernels = {}
        for name, (tot, n) in prof.items():
            if n == 0:
                continue
            avg_ms = tot / n
            ent = {"avg_ms": avg_ms, "launches_per_step": n / args.steps, "share": tot / total_k}
            if name in alg:
                bound, work = alg[name]
                if bound == "hbm":
                    a = work / (avg_ms * 1e-3) / 1e9
                    # algorithmic bytes against the HBM peak; the stick planes a z kernel exchanges with the plane kernel
                    # stay in L2 (the FFT path runs in L2-sized band chunks), so part of these bytes never reach DRAM:
                    # dram_bytes_ncu is what the committed ncu capture saw per launch
                    ent.update(bound="l2+hbm", achieved=a, peak=hbm_peak, unit="GB/s", frac=a / hbm_peak,
                               alg_bytes=work, dram_bytes_ncu=_ncu_traffic(cfg.name, name))
                else:
                    a = work / (avg_ms * 1e-3) / 1e12
                    ent.update(bound=bound, achieved=a, peak=dmma_peak, unit="TFLOP/s", frac=a / dmma_peak)
                    if name in effective:
                        ent["flops_per_complex_mac_executed"] = 6
                        ent["effective_tflops"] = effective[name] / (avg_ms * 1e-3) / 1e12
                if ent["frac"] > 1.0:
                    ent["invalid"] = "frac > 1: the work model or the peak is wrong"
            kernels[name] = ent
        if "k_plane" in kernels:
            # second roof of the fused plane kernel: the shared-memory pipe.  Algorithmic 16-byte accesses per z-plane (one
            # store + one load per element and exchange stage): y passes 6 N X, x passes N (4 N + 2 X);
            # peak = 128 B/clk/SM (B300_MICROARCH.md "smem crossbar BW") x SMs x the SM clock sampled during the run.
            n1 = cfg.grid[0]
            acc = cb * N3 * (8.0 * n1 * nx + 4.0 * n1 * n1)
            clk = (sampler.summary().get("sm_mhz") or 1965.0) * 1e6
            smem_peak = 128.0 * torch.cuda.get_device_properties(dev).multi_processor_count * clk / 1e12
            a = acc * 16.0 / (kernels["k_plane"]["avg_ms"] * 1e-3) / 1e12
            kernels["k_plane"]["co_bound"] = {"bound": "smem", "achieved": a, "peak": smem_peak, "unit": "TB/s",
                                              "frac": a / smem_peak,
                                              "note": "algorithmic shared-memory bytes of the six exchange stages per plane"}
        dom = max((k for k in kernels if "bound" in kernels[k]), key=lambda k: kernels[k]["share"])
        d = kernels[dom]
        roofline = {"kernel": dom, "bound": "hbm" if d["bound"] == "l2+hbm" else d["bound"], "achieved": d["achieved"], "peak": d["peak"],
                    "unit": d["unit"], "frac": d["frac"], "traffic": _ncu_traffic(cfg.name, dom),
                    "share_of_step": d["share"],
                    "peak_source": ("FP64 DMMA m8n8k4 register-resident probe run in this process; DMMA and DFMA "
                                    "share this issue budget (MEASURED_PEAKS.json has no FP64 entry)"
                                    if d["bound"] in ("tensor", "alu") else peak_src)}
        # the FFT / scatter / gather path as one HBM figure (north_star target >= 60 %)
        fft_ms = sum(kernels[k]["avg_ms"] for k in ("k_zinv", "k_plane", "k_zfwd") if k in kernels)
        fft_bytes = alg["k_zinv"][1] + alg["k_zfwd"][1] + cb * 2 * N3 * S * 16 + nvox * 8
        fft_path = {"achieved_GBps": fft_bytes / (fft_ms * 1e-3) / 1e9 if fft_ms else None, "peak_GBps": hbm_peak,
                    "frac": fft_bytes / (fft_ms * 1e-3) / 1e9 / hbm_peak if fft_ms else None,
                    "alg_bytes_per_call": fft_bytes, "ms_per_call": fft_ms, "peak_source": peak_src}
        # the same time charged with the bytes of the unfused one-pass-per-axis design (SURVEY 8(d) model D1: psi -> sticks,
        # sticks -> slab, slab -> x-FFT.V.x-FFT -> slab, slab -> sticks, sticks -> out): what an HBM-bound implementation
        # of the path would have to move; the north_star's ">= 60 % of HBM" refers to such passes
        slab = nx * cfg.grid[1] * N3 * 16
        d1_bytes = cb * (ng * 16 + N3 * S * 16 + (N3 * S * 16 + slab) + 2 * slab + (slab + N3 * S * 16)
                         + (N3 * S * 16 + 2 * ng * 16)) + nvox * 8
        fft_path["note"] = ("frac is on the bytes the fused path actually has to move (D2 model); the north_star's >= 60 % of HBM "
                            "is NOT met on those bytes: the fused plane kernel is bound by the FP64 pipe and shared memory, "
                            "see roofline / kernels.k_plane.  d1_model is a counterfactual (bytes of an unfused design)")
        fft_path["d1_model"] = {"counterfactual": True, "alg_bytes_per_call": d1_bytes,
                                "achieved_GBps": d1_bytes / (fft_ms * 1e-3) / 1e9 if fft_ms else None,
                                "frac": d1_bytes / (fft_ms * 1e-3) / 1e9 / hbm_peak if fft_ms else None}
        all_cfg = None
        if world == 1 and args.config == "cfg5" and not args.no_all_configs:
            sm_clk = (sampler.summary().get("sm_mhz") or 1965.0) * 1e6
            pk = (dmma_peak, 128.0 * torch.cuda.get_device_properties(dev).multi_processor_count * sm_clk / 1e12)
            all_cfg = {n: _small_config_figure(qm, torch, dev, n, args.steps, peaks=pk if n in ("cfg3", "cfg4") else None, hbm_peak=hbm_peak)
                       for n in ("cfg1", "cfg2", "cfg3", "cfg4")}
            all_cfg["cfg5"] = {"workload": _config_dict(cfg, ng, nsticks, nx)["workload"], "call_batch": cb,
                               "band_applies_per_s": value, "ms_per_full_band_apply": ms / args.steps,
                               "us_per_call": ms / args.steps * 1e3 / (cfg.nk * ((nb + cb - 1) // cb)),
                               "launch_mode": "calls", "launches_per_call": launches / args.steps / (cfg.nk * ((nb + cb - 1) // cb)),
                               "verified": verify["verified"] if verify else None}
        cpu = cpu_fft = None
        if world == 1 and not args.no_cpu_baseline:
            from oracle import gsphere as og    # cpu_baseline leg only
            miller, idx, g2 = og.gsphere(lat, cfg.ecutwfc_ry, cfg.grid, kpts[0])
            cpu = _cpu_oracle_rate(cfg, (lat, miller, g2, v, per_k[0][1], dblk, per_k[0][2]))
            cpu_fft = _cpu_fft_rate(cfg, (lat, miller, g2, v, per_k[0][1], dblk, per_k[0][2]), idx)
        n1g = cfg.grid[0]
        dens_tf = nb * N3 * ((nx + n1g) * 5.0 * n1g * np.log2(n1g) + 3.0 * n1g * cfg.grid[1]) / (density_ms * 1e-3) / 1e12
        so_flops = nb * (N3 * ((2 * nx + 2 * n1g) * 5.0 * n1g * np.log2(n1g) + 6.0 * n1g * cfg.grid[1])
                         + 2 * S * 5.0 * N3 * np.log2(N3) + 2 * 6.0 * ng)
        so_tf = so_flops / (splitop_ms * 1e-3) / 1e12
        ncalls_so = (nb + cb - 1) // cb
        so_bytes = cb * (ng * 16 + N3 * S * 16) + cb * 2 * N3 * S * 16 + cb * (N3 * S * 16 + ng * 16) + 2 * ng * 16 + nvox * 16
        so_gbps = so_bytes * ncalls_so / (splitop_ms * 1e-3) / 1e9
        tay_bytes = nb * ng * (32 + 3 * 64 + 48)
        tay_rest_ms = max(taylor_ms - 4 * ms / args.steps, 1e-6)
        tay_gbps = tay_bytes / (tay_rest_ms * 1e-3) / 1e9
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(3, args.warmup), "ms_per_step": ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "complex128", "data": "synthetic",
                "config": _config_dict(cfg, ng, nsticks, nx),
                "clocks": sampler.summary(),
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": bytes_io,
                        "d2h_bytes_per_step": bytes_io, "ms_per_step": ms_host / e2e_steps},
                "gpu_launches": int(launches),
                "verified": verify,
                "all_configs": all_cfg,
                "unfused_512_atoms": (_unfused_figure(qm, torch, dev, hbm_peak)
                                      if world == 1 and args.config == "cfg5" and not args.no_all_configs else None),
                "roofline": roofline, "fft_path": fft_path, "kernels": kernels,
                "fp64_peaks_tflops": {"dmma_probe": dmma_peak, "dfma_probe": dfma_peak},
                "one_call_all_bands": {"bands": nb, "ms": one_call_ms, "band_applies_per_s": nb / (one_call_ms * 1e-3)},
                "taylor": {"order": 4, "bands": nb, "call_batch": cb, "ms": taylor_ms,
                           "band_steps_per_s": nb / (taylor_ms * 1e-3),
                           "h_applies_per_s": 4 * nb / (taylor_ms * 1e-3),
                           # 4 applies + the r = 0 copy + 4 scale-and-accumulate launches per call; what is not the applies:
                           "apply_ms": 4 * ms / args.steps, "apply_share": 4 * (ms / args.steps) / taylor_ms,
                           "axpy": {"bound": "l2+hbm", "unit": "GB/s", "alg_bytes": tay_bytes, "ms": tay_rest_ms,
                                    "achieved": tay_gbps, "peak": hbm_peak, "frac": tay_gbps / hbm_peak,
                                    "note": "ms = taylor ms - 4 x the timed apply step; bytes = copy (32 B) + 3 x 64 B + 48 B "
                                            "per element; a 16-band block (20 MB) stays in L2 between the launches"}},
                "split_operator": {"bands": nb, "call_batch": cb, "ms": splitop_ms, "band_steps_per_s": nb / (splitop_ms * 1e-3),
                                   "launches_per_call": 3,
                                   # the same three kernels as the local part of an apply (k_zinv with the kinetic phase,
                                   # k_plane with a complex field, k_zfwd with the phase): both roofs of that path
                                   "bound": "alu", "unit": "TFLOP/s", "peak": dmma_peak, "achieved": so_tf, "frac": so_tf / dmma_peak,
                                   "hbm": {"alg_bytes_per_call": so_bytes, "achieved_GBps": so_gbps, "peak_GBps": hbm_peak,
                                           "frac": so_gbps / hbm_peak},
                                   "note": "flops: plane-kernel model with a complex multiply per voxel + the two z passes "
                                           "(5 n log2 n per stick) + the two phase multiplies"},
                "matrix_elements": {"nbra": n_me, "nket": n_me, "ecut_eps_ry": 10.0, "ng_eps": mtxel_ng, "ms": mtxel_ms,
                                    "pairs_per_s": n_me * n_me / (mtxel_ms * 1e-3), "bound": "hbm", "unit": "GB/s",
                                    "alg_bytes": (2 * n_me * n_me + 2 * n_me) * nvox * 16,
                                    "achieved": (2 * n_me * n_me + 2 * n_me) * nvox * 16 / (mtxel_ms * 1e-3) / 1e9,
                                    "peak": hbm_peak,
                                    "frac": (2 * n_me * n_me + 2 * n_me) * nvox * 16 / (mtxel_ms * 1e-3) / 1e9 / hbm_peak,
                                    "note": "bytes = two real-space boxes read per pair + one written per state"},
                "density": {"bands": nb, "call_batch": cb, "ms": density_ms, "bands_per_s": nb / (density_ms * 1e-3),
                            "bound": "alu", "unit": "TFLOP/s", "peak": dmma_peak,
                            "achieved": dens_tf, "frac": dens_tf / dmma_peak,
                            "note": "flops of the backward half of the plane kernel (y on X rows, x on N columns) + |psi|^2"},
                "subspace": {tag: {"na": n, "nb": n, "ng": ng, "ms": t_ms, "bound": "tensor",
                                   "achieved": 6.0 * n * n * ng / (t_ms * 1e-3) / 1e12, "peak": dmma_peak,
                                   "unit": "TFLOP/s", "frac": 6.0 * n * n * ng / (t_ms * 1e-3) / 1e12 / dmma_peak,
                                   "flops_per_complex_mac_executed": 6,
                                   "effective_tflops": 8.0 * n * n * ng / (t_ms * 1e-3) / 1e12}
                             for tag, (n, t_ms) in sub.items()},
                "cpu_baseline": cpu, "cpu_fft_baseline": cpu_fft}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cfg5")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-all-configs", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
