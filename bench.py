#!/usr/bin/env python
"""bench.py — coarse-op apply throughput on B200 (BASELINE.json metric: coarse-op site-updates/s
and effective HBM GB/s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2] [--impl ours|reference]

Workload (default C2 = BASELINE.json configs[1], the configuration the metric is quoted on):
16^3 x 24 periodic lattice, Nc = 48, complex64 links and vectors, 1 RHS, seeded Gamma-Hermitian
generator, "run with dagger=0 and dagger=1".  One STEP = one pass of the whole hot path over the
lattice in both modes: out = A.in followed by out2 = A^H.in (what one CGNE normal-equation
application does), i.e. 2 V site-updates.  `value` is device-timed with all inputs resident in HBM;
`e2e` goes through coarse_op_apply_host with pinned HOST vectors (H2D of the input vector and D2H
of the result inside the timed region; the links are operator state, set once, like weights).

N > 1 (torchrun): the path does not shard (north_star: single GPU, no inter-GPU communication), so
each rank runs an independent replica of the same workload; the timed region is bracketed by a
barrier + synchronize and the MAX over ranks is reported ("scaling": "weak").

`--impl reference`: there is no reference implementation for this paper (no code exists); the
reference arm times the CPU oracle (oracle/, fp64, as it stands) on the host cores on a bounded
sample of the same workload.  This and the `cpu_baseline` leg are the only places that execute
oracle/ outside tests.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

import synth

METRIC = "coarse-op site-updates/s"
UNIT = "site-updates/s"

def ncu_traffic_bytes(config: str, path: int, dagger: int, links: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, read from the newest
    `profiles/r*_ncu_traffic.csv` (written by `python -m paper_2212_12559_b200.ncu_summary` from the
    `ncu --set full` captures summarised beside it); None when that launch was not captured."""
    import csv
    import glob
    best = None
    for fn in sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_ncu_traffic.csv"))):
        try:
            with open(fn) as f:
                for row in csv.DictReader(f):
                    if (row["config"] == config and int(row["path"]) == path and int(row["dagger"]) == dagger
                            and row["links"] == links):
                        best = int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
        except Exception:
            continue
    return best


def compulsory_bytes_per_site(Nc: int, links: str, nrhs: int, hvec: bool = False) -> int:
    """SURVEY.md §8(d) / north_star: 9 Nc^2 link entries + 9 input vectors + 1 output vector.
    hvec: the 9 input vectors are int16 (re,im) + one fp32 norm per (site, rhs)."""
    link = 9 * Nc * Nc * (8 if links == "c64" else 4) + (36 if links == "i16" else 0)
    if hvec:
        return link + 9 * (Nc * nrhs * 4 + nrhs * 4) + Nc * nrhs * 8
    return link + 10 * Nc * nrhs * 8


def measured_peak_gbs():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.02):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self.power_w = []
        self._stop = threading.Event()
        self._thread = None
        self._period = period_s
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _loop(self):
        nv = self._nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                try:
                    self.power_w.append(nv.nvmlDeviceGetPowerUsage(self._h) / 1000.0)
                except Exception:
                    pass
                try:
                    mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
                except Exception:
                    mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(self._period)

    def __enter__(self):
        if self._nv is not None:
            self._thread = threading.Thread(target=self._loop, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thread is not None:
            self._thread.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        s = sorted(self.samples)
        out = {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
               "samples": len(s), "sm_mhz_min": s[0]}
        if self.power_w:
            pw = sorted(self.power_w)
            out["power_w"] = pw[len(pw) // 2]
            out["power_w_max"] = pw[-1]
        return out


def dist_env():
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return world, rank, local


def reduce_max_sum(local_ms: float, local_units: float, device=None):
    """(max over ranks of the elapsed time, sum over ranks of the units processed)."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local_ms, local_units
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


# ------------------------------------------------------------------------------- CPU oracle legs
def oracle_sample_dims(cfg):
    """Bounded sample of the workload for the CPU oracle: a slab of the same lattice (same Nc, same
    generator, same per-site work), periodic on its own."""
    d = list(cfg["dims"])
    per_site = 9 * cfg["Nc"] ** 2 * cfg["nrhs"]
    budget = 4.0e7 * 1.0            # complex MACs per apply (~0.05-0.5 s on 8-64 host cores)
    # halve the currently LONGEST extent (last index first) while over budget: extents stay >= 4 as long as
    # possible, so x+mu and x-mu remain distinct sites as in the workload (two extent-2 directions would be
    # friendlier to the CPU caches than the real lattice)
    while d[0] * d[1] * d[2] * d[3] * per_site > budget and max(d) > 2:
        mu = max(range(4), key=lambda k: (d[k], k))
        d[mu] = max(2, d[mu] // 2)
    return tuple(d)


def make_oracle_sample(cfg, device):
    import oracle
    dims = oracle_sample_dims(cfg)
    Nc, nrhs = cfg["Nc"], cfg["nrhs"]
    links = synth.make_gamma_hermitian_links(dims, Nc, cfg["seed"], device=device).cpu().numpy()
    scales, prec = None, oracle.LINK_C64
    if cfg["links"] == "i16":
        q, scales = oracle.quantize_i16(links, Nc)
        links, prec = q.reshape(-1, 9, Nc, Nc, 2), oracle.LINK_I16
    vin = synth.make_vectors(dims, Nc, nrhs, cfg["seed"] + 1, device=device).cpu().numpy()
    return dims, links, scales, prec, vin


def oracle_step(sample, cfg, daggers, nthreads=0):
    import oracle
    dims, links, scales, prec, vin = sample
    for dg in daggers:
        oracle.coarse_apply(dims, cfg["Nc"], links, vin, nrhs=cfg["nrhs"], dagger=dg,
                            link_precision=prec, scales=scales, nthreads=nthreads)


def time_oracle(cfg, daggers, device, min_seconds=10.0, max_steps=100000, nthreads=0):
    import oracle
    oracle.build()
    sample = make_oracle_sample(cfg, device)
    V = synth.lattice_volume(sample[0])
    oracle_step(sample, cfg, daggers, nthreads)            # warm-up (page-in, thread pool)
    t0 = time.perf_counter()
    n = 0
    while n < max_steps and (time.perf_counter() - t0 < min_seconds or n < 3):
        oracle_step(sample, cfg, daggers, nthreads)
        n += 1
    dt = time.perf_counter() - t0
    return {
        "value": V * len(daggers) * n / dt,
        "unit": UNIT,
        "cores": nthreads if nthreads > 0 else oracle.max_threads(),
        "kind": "oracle",
        "sample": f"{n} steps on a {'x'.join(map(str, sample[0]))} slab of the workload lattice "
                  f"({V} sites, same Nc/links/nrhs/generator, periodic on its own), {dt:.1f} s of CPU time",
    }


def run_reference(args, cfg, daggers):
    """--impl reference: the CPU oracle as it stands, on the host cores (rank 0 only)."""
    world, rank, _ = dist_env()
    if rank != 0:
        return 0
    import oracle
    oracle.build()
    device = "cuda" if torch.cuda.is_available() else "cpu"
    sample = make_oracle_sample(cfg, device)
    V = synth.lattice_volume(sample[0])
    for _ in range(args.warmup):
        oracle_step(sample, cfg, daggers)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_step(sample, cfg, daggers)
    dt = time.perf_counter() - t0
    value = V * len(daggers) * args.steps / dt
    sample_desc = (f"each step = dagger {daggers} applies on a {'x'.join(map(str, sample[0]))} slab "
                   f"({V} sites) of the workload lattice, same Nc/links/nrhs/generator")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": workload_name(args.config, cfg), "sample": sample_desc},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
                         "sample": sample_desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def workload_name(name, cfg, hvec=False):
    return (f"{name}: coarse-op apply, {'x'.join(map(str, cfg['dims']))} periodic lattice, Nc={cfg['Nc']}, "
            f"{cfg['links']} links, {'int16+norm input / complex64 output' if hvec else 'complex64'} vectors, "
            f"nrhs={cfg['nrhs']}")


# ------------------------------------------------------------------------------- in-run parity
def parity_sample_sites(dims, n_random, seed):
    """Corners, first/last sites and seeded random sites of the lattice (sorted, unique)."""
    L0, L1, L2, L3 = dims
    V = L0 * L1 * L2 * L3
    pts = [0, 1 % V, V - 2 if V > 1 else 0, V - 1]
    for x3 in (0, L3 - 1):
        for x2 in (0, L2 - 1):
            for x1 in (0, L1 - 1):
                for x0 in (0, L0 - 1):
                    pts.append(x0 + L0 * (x1 + L1 * (x2 + L2 * x3)))
    rnd = np.random.default_rng(seed).integers(0, V, size=n_random)
    return np.unique(np.concatenate([np.asarray(pts, dtype=np.int64), rnd])).astype(np.int64)


def parity_check(cfg, links, scales, vin, outs, n_random=64, hvec=None):
    """"parity is checked in the same run, before timing, on the same buffers".  The device
    buffers the timed loop is about to use hold one apply per dagger; the CPU oracle (its per-site
    evaluation, `oracle.coarse_apply_sites`) recomputes >= 64 sampled output sites from the links and
    vectors those sites touch.  Returns the worst relative L2 error over daggers and right-hand sides.
    `hvec` = (int16 vector, norms): the run applies the operator to half-precision vectors (--hvec), and the oracle
    evaluates the same int16 + norm arrays.
    (Part of the oracle legs of this script, like cpu_baseline: the product path never calls it.)"""
    import oracle
    oracle.build()
    dims, Nc, nrhs = cfg["dims"], cfg["Nc"], cfg["nrhs"]
    V = synth.lattice_volume(dims)
    i16 = cfg["links"] == "i16"
    sites = parity_sample_sites(dims, n_random, cfg["seed"])
    need = np.unique(np.concatenate([oracle.neighbours(dims, int(s)) for s in sites]))
    flat = links if i16 else torch.view_as_real(links)
    links_h = np.empty((V, 9, Nc, Nc, 2), dtype=np.int16 if i16 else np.float32)   # only the needed sites are touched
    idx = torch.as_tensor(need, device=flat.device)
    links_h[need] = flat[idx].cpu().numpy().reshape(len(need), 9, Nc, Nc, 2)
    scales_h = None if scales is None else scales.cpu().numpy()
    vin_h = vin.cpu().numpy() if hvec is None else None
    hq_h, hn_h = (hvec[0].cpu().numpy(), hvec[1].cpu().numpy()) if hvec is not None else (None, None)
    worst, worst_site = 0.0, 0.0
    sidx = torch.as_tensor(sites, device=flat.device)
    for dg, out in outs.items():
        if hvec is not None:
            ref = oracle.coarse_apply_hvec_sites(dims, Nc, links_h, hq_h, hn_h, sites, nrhs=nrhs, dagger=dg,
                                                 link_precision=oracle.LINK_I16 if i16 else oracle.LINK_C64, scales=scales_h)
        else:
            ref = oracle.coarse_apply_sites(dims, Nc, links_h, vin_h, sites, nrhs=nrhs, dagger=dg,
                                            link_precision=oracle.LINK_I16 if i16 else oracle.LINK_C64, scales=scales_h)
        got = out[sidx].cpu().numpy().astype(np.complex128)
        for r in range(nrhs):
            worst = max(worst, float(np.linalg.norm(got[..., r] - ref[..., r]) / np.linalg.norm(ref[..., r])))
        per_site = np.linalg.norm((got - ref).reshape(len(sites), -1), axis=1) / np.linalg.norm(ref.reshape(len(sites), -1), axis=1)
        worst_site = max(worst_site, float(per_site.max()))
    return {"rel_l2": worst, "worst_site_rel_l2": worst_site, "sites": int(len(sites)), "tolerance": 1e-5,
            "ok": bool(worst <= 1e-5 and worst_site <= 5e-5)}


def measure_config(name, steps, local, dev, read_ceiling=None, override=None):
    """One BASELINE config on the AUTO path: in-run parity on sampled sites, then `steps` applies per dagger
    timed with CUDA events (L2-resident lattices: one CUDA graph per dagger, warm, plus a cold number over
    rotating link copies).  Sub-record of the default bench line (`configs`; `override` changes links / nrhs
    for the `extras` records)."""
    import paper_2212_12559_b200 as cop
    cfg = synth.config(name)
    cfg.update(override or {})
    dims, Nc, nrhs = cfg["dims"], cfg["Nc"], cfg["nrhs"]
    V = synth.lattice_volume(dims)
    prec = cop.LINK_I16 if cfg["links"] == "i16" else cop.LINK_C64
    links = synth.make_gamma_hermitian_links(dims, Nc, cfg["seed"], device=dev)
    scales = None
    if prec == cop.LINK_I16:
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device=dev)
        scales = torch.empty((V, 9), dtype=torch.float32, device=dev)
        cop.coarse_op_quantize_i16(links, Nc, q, scales)
        torch.cuda.synchronize()
        links = q
    vin = synth.make_vectors(dims, Nc, nrhs, cfg["seed"] + 1, device=dev)
    outs = {dg: torch.full_like(vin, float("nan")) for dg in (0, 1)}
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
    stream = torch.cuda.current_stream()
    hvec = bool(cfg.get("hvec"))        # half-precision input vectors: int16 + per-site norm
    vq = vnorm = None
    if hvec:
        vq = torch.empty((V, Nc, nrhs, 2), dtype=torch.int16, device=dev)
        vnorm = torch.empty((V, nrhs), dtype=torch.float32, device=dev)
        cop.coarse_op_quantize_vec_i16(vin, Nc, nrhs, vq, vnorm)

    def apply(o, out, dg):
        if hvec:
            o.apply_hvec(vq, vnorm, out, nrhs=nrhs, dagger=dg)
        else:
            o.apply(vin, out, nrhs=nrhs, dagger=dg)

    for dg in (0, 1):
        apply(op, outs[dg], dg)
    torch.cuda.synchronize()
    path = op.last_path
    parity = parity_check(cfg, links, scales, vin, outs, hvec=(vq, vnorm) if hvec else None)
    link_bytes = links.numel() * links.element_size()
    l2_bytes = torch.cuda.get_device_properties(dev).L2_cache_size
    bps = compulsory_bytes_per_site(Nc, cfg["links"], nrhs, hvec)
    peak, _ = measured_peak_gbs()
    rec = {"workload": workload_name(name, cfg, hvec), "path": path, "steps": steps, "parity": parity,
           "algorithmic_bytes_per_launch": bps * V}

    def graph_of(fn):
        g = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.graph(g, stream=side):
            fn()
        torch.cuda.current_stream().wait_stream(side)
        g.replay()
        torch.cuda.synchronize()
        return g

    def time_graph(g):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        g.replay()
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b)

    with ClockSampler(local) as clocks:
        if link_bytes <= 2 * l2_bytes:
            reps = max(steps, 400)          # a graph launch costs tens of us: amortise it over many 6-10 us applies
            warm = {dg: time_graph(graph_of(lambda dg=dg: [apply(op, outs[dg], dg) for _ in range(reps)])) / reps
                    for dg in (0, 1)}
            n_copies = int(3 * l2_bytes // max(1, link_bytes)) + 2
            copies = [(links.clone(), None if scales is None else scales.clone()) for _ in range(n_copies)]
            ops = [cop.CoarseOp(dims, Nc, prec).set_links(l, sc).set_option(cop.OPT_KEEP_LINKS, 1) for l, sc in copies]
            creps = max(reps, 2 * n_copies)
            ms = {dg: time_graph(graph_of(lambda dg=dg: [apply(ops[r % n_copies], outs[dg], dg)
                                                         for r in range(creps)])) / creps for dg in (0, 1)}
            for o in ops:
                o.close()
            del ops, copies
            rec["timing"] = "CUDA graph of %d applies per dagger; ms = COLD (links rotated over %d copies > L2), warm-L2 beside" % (creps, n_copies)
            rec["warm_l2_ms"] = {str(dg): warm[dg] for dg in (0, 1)}
        else:
            for _ in range(3):
                for dg in (0, 1):
                    apply(op, outs[dg], dg)
            ev = {dg: [] for dg in (0, 1)}
            for _ in range(steps):
                for dg in (0, 1):
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record(stream)
                    apply(op, outs[dg], dg)
                    b.record(stream)
                    ev[dg].append((a, b))
            torch.cuda.synchronize()
            ms = {dg: sum(a.elapsed_time(b) for a, b in ev[dg]) / steps for dg in (0, 1)}
            rec["timing"] = "CUDA events around each of %d applies per dagger (dagger 0 / 1 alternating), mean" % steps
    rec["ms"] = {str(dg): ms[dg] for dg in (0, 1)}
    rec["gbs"] = {str(dg): bps * V / (ms[dg] * 1e-3) / 1e9 for dg in (0, 1)}
    rec["frac"] = {str(dg): rec["gbs"][str(dg)] / peak for dg in (0, 1)}
    rec["frac_of_nominal_8000"] = {str(dg): rec["gbs"][str(dg)] / 8000.0 for dg in (0, 1)}
    if read_ceiling:
        rec["frac_of_read_ceiling"] = {str(dg): rec["gbs"][str(dg)] / read_ceiling for dg in (0, 1)}
    rec["msite_updates_per_s"] = {str(dg): V / (ms[dg] * 1e-3) / 1e6 for dg in (0, 1)}
    rec["clocks"] = clocks.summary()
    rec["traffic"] = None if override else {str(dg): ncu_traffic_bytes(name, path, dg, cfg["links"]) for dg in (0, 1)}
    op.close()
    return rec


# ------------------------------------------------------------------------------- GPU arm
def run_ours(args, cfg, daggers):
    import paper_2212_12559_b200 as cop

    world, rank, local = dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the coarse-op library has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    dims, Nc, nrhs = cfg["dims"], cfg["Nc"], cfg["nrhs"]
    V = synth.lattice_volume(dims)
    prec = cop.LINK_I16 if cfg["links"] == "i16" else cop.LINK_C64

    links = synth.make_gamma_hermitian_links(dims, Nc, cfg["seed"], device=dev)
    scales = None
    if prec == cop.LINK_I16:
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device=dev)
        scales = torch.empty((V, 9), dtype=torch.float32, device=dev)
        cop.coarse_op_quantize_i16(links, Nc, q, scales)
        torch.cuda.synchronize()
        links = q
        del q
    vin = synth.make_vectors(dims, Nc, nrhs, cfg["seed"] + 1, device=dev)
    vouts = [torch.empty_like(vin) for _ in daggers]
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
    if args.path:
        op.set_option(cop.OPT_PATH, args.path)
    if args.stages:
        op.set_option(cop.OPT_STAGES, args.stages)
    if args.grid:
        op.set_option(cop.OPT_GRID, args.grid)
    if args.fine:
        op.set_option(cop.OPT_FINE, args.fine)
    if args.keep_links:
        op.set_option(cop.OPT_KEEP_LINKS, args.keep_links)
    if args.pdl:
        op.set_option(cop.OPT_PDL, args.pdl)
    if args.warp_items:
        op.set_option(cop.OPT_WARP_ITEMS, args.warp_items)
    if args.tensor_i8:
        op.set_option(cop.OPT_TENSOR_I8, args.tensor_i8)

    vq = vnorm = None
    if args.hvec:
        vq = torch.empty((V, Nc, nrhs, 2), dtype=torch.int16, device=dev)
        vnorm = torch.empty((V, nrhs), dtype=torch.float32, device=dev)
        cop.coarse_op_quantize_vec_i16(vin, Nc, nrhs, vq, vnorm)
        torch.cuda.synchronize()

    oq = onorm = None
    if args.hout:
        oq = torch.empty((V, Nc, nrhs, 2), dtype=torch.int16, device=dev)
        onorm = torch.empty((V, nrhs), dtype=torch.float32, device=dev)

    def apply_one(out, dg):
        if args.hout:
            op.apply_hout(vq if args.hvec else vin, vnorm if args.hvec else None, out, oq, onorm, nrhs=nrhs, dagger=dg)
        elif args.hvec:
            op.apply_hvec(vq, vnorm, out, nrhs=nrhs, dagger=dg)
        else:
            op.apply(vin, out, nrhs=nrhs, dagger=dg)

    stream = torch.cuda.current_stream()
    launches = 0
    link_bytes = links.numel() * links.element_size()
    l2_bytes = torch.cuda.get_device_properties(dev).L2_cache_size
    # A lattice whose links fit L2 takes microseconds per apply: per-launch host overhead (Python +
    # ctypes + launch, ~10 us) would be what is timed.  Such configs are timed as ONE CUDA graph of
    # all K steps (coarse_op_apply is capturable: it only enqueues).
    use_graph = args.graph == "on" or (args.graph == "auto" and link_bytes <= 2 * l2_bytes)

    path_of = {}

    def step(record=None):
        nonlocal launches
        for k, dg in enumerate(daggers):
            if record is not None:
                e0 = torch.cuda.Event(enable_timing=True)
                e1 = torch.cuda.Event(enable_timing=True)
                e0.record(stream)
            apply_one(vouts[k], dg)
            launches += op.last_launches
            path_of[dg] = op.last_path              # AUTO may pick another family per mode (complex64, 4 RHS)
            if record is not None:
                e1.record(stream)
                record[dg].append((e0, e1))

    def capture(fn):
        g = torch.cuda.CUDAGraph()
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.graph(g, stream=side):
            fn()
        torch.cuda.current_stream().wait_stream(side)
        return g

    def time_graph(g):
        g.replay()                                   # warm-up replay (instantiation, L2 state)
        torch.cuda.synchronize()
        a = torch.cuda.Event(enable_timing=True)
        b = torch.cuda.Event(enable_timing=True)
        a.record(stream)
        g.replay()
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    # parity in the same run, before timing, on the buffers the timed loop writes
    parity = None
    if rank == 0 and not args.no_parity:      # (with --hout the complex64 result is what is checked)
        parity = parity_check(cfg, links, scales, vin, {dg: vouts[k] for k, dg in enumerate(daggers)},
                              hvec=(vq, vnorm) if args.hvec else None)
        if not parity["ok"]:
            raise RuntimeError("bench.py: the GPU result does not match the CPU oracle on the sampled sites: %r" % (parity,))
    barrier()
    cold = None
    if use_graph:
        launches = 0
        g_steps = capture(lambda: [step() for _ in range(args.steps)])
        gpu_launches = launches
        g_one = {dg: capture(lambda dg=dg, i=i: [apply_one(vouts[i], dg)
                                             for _ in range(args.steps)])
                 for i, dg in enumerate(daggers)}
        barrier()
        with ClockSampler(local) as clocks:
            local_ms = time_graph(g_steps)
            kernel_ms = {dg: time_graph(g_one[dg]) / args.steps for dg in daggers}
        barrier()
        # cold number: rotate over enough distinct link copies that every apply reads from DRAM
        n_copies = int(3 * l2_bytes // max(1, link_bytes)) + 2
        if n_copies * link_bytes <= 24e9:
            copies = [(links.clone(), None if scales is None else scales.clone()) for _ in range(n_copies)]
            ops = [cop.CoarseOp(dims, Nc, prec).set_links(l, sc) for l, sc in copies]
            for o in ops:
                o.set_option(cop.OPT_KEEP_LINKS, 1)
            reps = max(args.steps, 2 * n_copies)
            g_cold = {dg: capture(lambda dg=dg: [ops[r % n_copies].apply(vin, vouts[i], nrhs=nrhs, dagger=dg)
                                                 for r in range(reps)])
                      for i, dg in enumerate(daggers)}
            cold = {"copies": n_copies, "kernel_ms": {str(dg): time_graph(g_cold[dg]) / reps for dg in daggers}}
            del g_cold
            for o in ops:
                o.close()
            del ops, copies
    else:
        barrier()
        launches = 0
        per_launch = {dg: [] for dg in daggers}
        t_start = torch.cuda.Event(enable_timing=True)
        t_end = torch.cuda.Event(enable_timing=True)
        with ClockSampler(local) as clocks:
            torch.cuda.synchronize()
            t_start.record(stream)
            for _ in range(args.steps):
                step(per_launch)
            t_end.record(stream)
            torch.cuda.synchronize()
        barrier()
        local_ms = t_start.elapsed_time(t_end)
        gpu_launches = launches
        kernel_ms = {dg: sum(a.elapsed_time(b) for a, b in per_launch[dg]) / max(1, len(per_launch[dg]))
                     for dg in daggers}
    units_local = float(V) * len(daggers) * args.steps
    total_ms, units = reduce_max_sum(local_ms, units_local, device=dev)
    value = units / (total_ms * 1e-3)

    # pure-read ceiling of this GPU for the apply's access pattern (the library's TMA-ring probe over
    # the link array itself), context for the roofline fraction: a copy-based peak is half writes
    read_ceiling = None
    if link_bytes > 4 * l2_bytes:
        best = 0.0
        for stg in (5, 6, 7):
            cop.coarse_op_probe_read(links, 16384, stg)
            a = torch.cuda.Event(enable_timing=True)
            b = torch.cuda.Event(enable_timing=True)
            a.record(stream)
            nb = 0
            for _ in range(3):
                nb += cop.coarse_op_probe_read(links, 16384, stg)
            b.record(stream)
            torch.cuda.synchronize()
            best = max(best, nb / (a.elapsed_time(b) * 1e-3) / 1e9)
        read_ceiling = best


    # ---- end to end: host vectors through coarse_op_apply_host
    vin_h = vin.cpu().pin_memory()
    vout_h = torch.empty_like(vin_h).pin_memory()
    e2e_steps = max(3, min(args.steps, 20))
    for dg in daggers:
        op.apply_host(vin_h, vout_h, nrhs=nrhs, dagger=dg)
    torch.cuda.synchronize()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        for dg in daggers:
            op.apply_host(vin_h, vout_h, nrhs=nrhs, dagger=dg)      # synchronises the stream itself
    torch.cuda.synchronize()
    e2e_ms_local = 1e3 * (time.perf_counter() - t0)
    barrier()
    e2e_ms, e2e_units = reduce_max_sum(e2e_ms_local, float(V) * len(daggers) * e2e_steps, device=dev)
    vec_bytes = V * Nc * nrhs * 8

    if rank != 0:
        return 0

    peak, peak_src = measured_peak_gbs()
    bps = compulsory_bytes_per_site(Nc, cfg["links"], nrhs, args.hvec)
    dom = daggers[0]
    achieved = bps * V / (kernel_ms[dom] * 1e-3) / 1e9
    roofline = {
        "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
        "traffic": None if args.hvec else ncu_traffic_bytes(args.config, path_of.get(dom, op.last_path), dom, cfg["links"]),
        "kernel": "coarse_apply_%s<Nc=%d,%s,dagger=%d%s>" % (
            {cop.PATH_SIMPLE: "simple", cop.PATH_STREAM: "stream", cop.PATH_TENSOR: "tensor",
             cop.PATH_BLOCK: "block"}.get(path_of.get(dom, op.last_path), "?"), Nc, "i16" if prec else "c64", dom,
            "" if nrhs == 1 else ",nrhs=%d" % nrhs),
        "kernel_ms": kernel_ms[dom],
        "algorithmic_bytes_per_launch": bps * V,
        "peak_source": peak_src,
        "frac_of_nominal_8000": achieved / 8000.0,
    }
    if read_ceiling is not None:
        roofline["read_ceiling_gbs"] = read_ceiling
        roofline["frac_of_read_ceiling"] = achieved / read_ceiling
        roofline["read_ceiling_note"] = ("coarse_op_probe_read: the same TMA ring with an idle consumer, 16 KB stages, "
                                         "best of 5-7 stages, over the link array, measured in this run")
    for dg in daggers[1:]:
        roofline[f"dagger{dg}_achieved"] = bps * V / (kernel_ms[dg] * 1e-3) / 1e9
        roofline[f"dagger{dg}_kernel_ms"] = kernel_ms[dg]
    if use_graph:
        roofline["timing"] = "one CUDA graph of K applies per dagger, time / K"
        if link_bytes <= l2_bytes:
            # L2-resident lattice: back-to-back applies never touch DRAM, so the HBM fraction is quoted
            # on the COLD number (rotating link copies); the warm time is kept beside it.
            roofline["warm_l2_kernel_ms"] = {str(dg): kernel_ms[dg] for dg in daggers}
            if cold is not None:
                roofline["kernel_ms"] = cold["kernel_ms"][str(dom)]
                roofline["achieved"] = bps * V / (roofline["kernel_ms"] * 1e-3) / 1e9
                roofline["frac"] = roofline["achieved"] / peak
                roofline["frac_of_nominal_8000"] = roofline["achieved"] / 8000.0
                roofline["cold"] = cold
                roofline["note"] = "achieved/frac are COLD (links rotated over %d copies > L2); warm-L2 times beside" % cold["copies"]

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {
            "workload": workload_name(args.config, cfg, args.hvec),
            "step": f"one apply per dagger in {daggers} (2V site-updates)" if len(daggers) == 2 else f"one apply, dagger={daggers[0]}",
            "l2": "inputs larger than L2 (links %.2f GB per apply, no flush needed)" % (links.numel() * links.element_size() / 1e9)
                  if link_bytes > 4 * 126e6 else "working set fits L2: `value` is the warm-L2 number (CUDA graph of all K steps); roofline quotes the cold one",
            "multi_gpu": "replicas only (the path does not shard; no collective)",
            "seed": cfg["seed"],
        },
        "effective_gbs": value * bps / 1e9,
        "clocks": clocks.summary(),
        "e2e": {"value": e2e_units / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": vec_bytes * len(daggers),
                "d2h_bytes_per_step": vec_bytes * len(daggers), "steps": e2e_steps,
                "note": "vectors from/to pinned host memory every apply; links are resident operator state"},
        "gpu_launches": gpu_launches,
        "roofline": roofline,
    }
    if parity is not None:
        line["parity"] = parity
    op.close()
    del links, vin, vouts, op
    if scales is not None:
        del scales
    torch.cuda.empty_cache()
    # The other BASELINE configs as sub-records of the default line (the driver runs one line): AUTO path,
    # in-run parity, 20 applies per dagger each.  Their launches are not part of `gpu_launches`/`value`.
    if world == 1 and args.all_configs and args.config == "C2" and not args.hvec:
        line["configs"] = {}
        for name in ("C1", "C3", "C4", "C5"):
            line["configs"][name] = measure_config(name, args.config_steps, local, dev, read_ceiling)
            torch.cuda.empty_cache()
        # the paper's storage format (int16 links) with several right-hand sides (its future work, L200;
        # 3 = one propagator): not BASELINE configs, reported beside them
        line["extras"] = {}
        for key, name, ov in (("C5_int16_nrhs16", "C5", {"links": "i16"}), ("C5_int16_nrhs3", "C5", {"links": "i16", "nrhs": 3}),
                              ("C4_nrhs3", "C4", {"nrhs": 3}),
                              # ... and with the paper's half-precision VECTORS too (L97): both operands 16-bit fixed point
                              ("C5_int16_hvec_nrhs16", "C5", {"links": "i16", "hvec": True}),
                              ("C4_hvec_nrhs3", "C4", {"nrhs": 3, "hvec": True}),
                              # the paper's own per-GPU coarse volumes (PAPER.md:L117/L125/L133): level 2 and level 3, int16
                              ("P2_paper_level2_per_gpu", "P2", None), ("P3_paper_level3_per_gpu", "P3", None)):
            line["extras"][key] = measure_config(name, args.config_steps, local, dev, read_ceiling, override=ov)
            torch.cuda.empty_cache()
        # the SURVEY.md §8(f) rows on the C3 shape (the paper's level-2 operator): the even/odd Schur-hat operator (f1), one
        # CA-GCR(8) smoother cycle (f3), and the device build of the block-preconditioned links on C1's lattice (f1)
        sub = argparse.Namespace(**vars(args))
        sub.steps, sub.warmup, sub.cheb = 10, 3, False
        for key, fn, cname in (("schur_C3", run_schur, "C3"), ("cagcr8_C3", run_cagcr, "C3"), ("hat_links_C1", run_hat, "C1")):
            rec = fn(sub, synth.config(cname), emit=False)
            line["extras"][key] = {k: rec[k] for k in ("metric", "value", "unit", "ms_per_step", "config", "clocks", "gpu_launches",
                                                       "roofline", "cagcr", "parity") if k in rec}
            torch.cuda.empty_cache()
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = time_oracle(cfg, daggers, dev, min_seconds=args.cpu_seconds)
        if args.all_configs and args.config == "C2":
            # "plus a 1-thread number on C1 and C3"
            line["cpu_baseline"]["one_thread"] = {
                name: time_oracle(synth.config(name), daggers, dev, min_seconds=2.0, nthreads=1) for name in ("C1", "C3")}
    print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return 0


# ------------------------------------------------------------------------------- even/odd workload
def run_schur(args, cfg, emit=True):
    """--workload schur (not the default bench line): the left-preconditioned
    Schur operator on block-preconditioned links, Shat_e v = v - Dhat_eo Dhat_oe v, and its adjoint.
    One step = Shat_e.v then Shat_e^H.v = 4 parity-restricted hop launches of V/2 sites each."""
    import paper_2212_12559_b200 as cop
    world, rank, local = dist_env()
    if world > 1:
        raise RuntimeError("--workload schur is a single-GPU measurement")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dims, Nc = cfg["dims"], cfg["Nc"]
    V = synth.lattice_volume(dims)
    prec = cop.LINK_I16 if cfg["links"] == "i16" else cop.LINK_C64
    links = synth.make_arbitrary_links(dims, Nc, cfg["seed"], device=dev)      # stands in for Yhat = X^-1 Y
    scales = None
    if prec == cop.LINK_I16:
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device=dev)
        scales = torch.empty((V, 9), dtype=torch.float32, device=dev)
        cop.coarse_op_quantize_i16(links, Nc, q, scales)
        torch.cuda.synchronize()
        links = q
    v = synth.make_vectors(dims, Nc, 1, cfg["seed"] + 1, device=dev)
    t, out = torch.zeros_like(v), torch.zeros_like(v)
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
    stream = torch.cuda.current_stream()

    def schur(dagger):
        op.apply_parts(None, v, t, dagger=dagger, parity=cop.PARITY_ODD, local=cop.LOCAL_NONE, alpha=0.0, beta=1.0)
        op.apply_parts(v, t, out, dagger=dagger, parity=cop.PARITY_EVEN, local=cop.LOCAL_IDENTITY, alpha=1.0, beta=-1.0)

    for _ in range(max(args.warmup, 3)):
        schur(0); schur(1)
    torch.cuda.synchronize()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    with ClockSampler(local) as clocks:
        for e in ev:
            e[0].record(stream); schur(0); e[1].record(stream); schur(1); e[2].record(stream)
        torch.cuda.synchronize()
    total_ms = ev[0][0].elapsed_time(ev[-1][2])
    ms0 = sum(e[0].elapsed_time(e[1]) for e in ev) / args.steps
    ms1 = sum(e[1].elapsed_time(e[2]) for e in ev) / args.steps
    link_site = 8 * Nc * Nc * (8 if prec == cop.LINK_C64 else 4) + (32 if prec == cop.LINK_I16 else 0)
    bytes_schur = (V // 2) * (2 * link_site + (8 + 1 + 8 + 1 + 1) * Nc * 8)     # hop: 8 reads + 1 write; xpay hop: + u
    peak, peak_src = measured_peak_gbs()
    line = {
        "metric": METRIC, "value": 2.0 * V * args.steps / (total_ms * 1e-3), "unit": UNIT, "n_gpus": 1,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "even/odd Schur-hat operator (v - Dhat_eo Dhat_oe v) and its adjoint on the %s lattice, "
                               "Nc=%d, %s links: 4 parity-restricted hop launches of V/2 sites per step" %
                               ("x".join(map(str, dims)), Nc, cfg["links"]), "seed": cfg["seed"]},
        "clocks": clocks.summary(), "gpu_launches": 4 * args.steps,
        "roofline": {"bound": "hbm", "achieved": bytes_schur / (ms0 * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                     "frac": bytes_schur / (ms0 * 1e-3) / 1e9 / peak, "traffic": None, "peak_source": peak_src,
                     "kernel": "2 x coarse_apply_stream<GEN> (hop to odd, identity - hop to even)",
                     "schur_ms": ms0, "schur_dagger_ms": ms1, "algorithmic_bytes_per_schur_apply": bytes_schur,
                     "dagger_achieved": bytes_schur / (ms1 * 1e-3) / 1e9},
    }
    if not emit:
        op.close()
        return line
    print(json.dumps(line), flush=True)
    op.close()
    return 0


def run_hat(args, cfg, emit=True):
    """--workload hat: build the block-preconditioned links
    Yhat_m = X^-1 Y_m of the config's operator on the device (coarse_op_build_hat_links) and quantise them
    to int16 when the config stores int16 links.  A set-up step: one step = one build over the lattice.
    Bound by fp64 FMA throughput (72 Nc^3 flops per site), not HBM; both fractions are reported."""
    import paper_2212_12559_b200 as cop
    world, rank, local = dist_env()
    if world > 1:
        raise RuntimeError("--workload hat is a single-GPU measurement")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dims, Nc = cfg["dims"], cfg["Nc"]
    V = synth.lattice_volume(dims)
    links = synth.make_gamma_hermitian_links(dims, Nc, cfg["seed"], device=dev)
    op = cop.CoarseOp(dims, Nc, cop.LINK_C64).set_links(links)
    hat = torch.empty_like(links)
    info = torch.zeros((1,), dtype=torch.int32, device=dev)
    work = op.build_hat_links(hat, info=info)
    torch.cuda.synchronize()
    parity = None
    if not args.no_parity:
        import oracle
        sites = parity_sample_sites(dims, 24, cfg["seed"])
        ref = oracle.hat_links(links[torch.as_tensor(sites, device=dev)].cpu().numpy())
        got = hat[torch.as_tensor(sites, device=dev)].cpu().numpy().astype(np.complex128)
        err = np.linalg.norm((got - ref).reshape(len(sites), 9, -1), axis=2) / np.linalg.norm(ref.reshape(len(sites), 9, -1), axis=2)
        parity = {"rel_l2_per_matrix_max": float(err.max()), "sites": int(len(sites)), "tolerance": 1e-6,
                  "ok": bool(err.max() <= 1e-6), "singular_sites": int(info.item())}
        if not parity["ok"]:
            raise RuntimeError("bench.py --workload hat: device-built hat links differ from the oracle: %r" % (parity,))
    stream = torch.cuda.current_stream()
    q = sc = None
    if cfg["links"] == "i16":
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device=dev)
        sc = torch.empty((V, 9), dtype=torch.float32, device=dev)

    def step():
        op.build_hat_links(hat, work=work)
        if q is not None:
            cop.coarse_op_quantize_i16(hat, Nc, q, sc)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    steps = min(args.steps, 20)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(steps)]
    with ClockSampler(local) as clocks:
        for a, b, c in ev:
            a.record(stream)
            op.build_hat_links(hat, work=work)
            b.record(stream)
            if q is not None:
                cop.coarse_op_quantize_i16(hat, Nc, q, sc)
            c.record(stream)
        torch.cuda.synchronize()
    ms_build = sum(a.elapsed_time(b) for a, b, c in ev) / steps
    ms_total = sum(a.elapsed_time(c) for a, b, c in ev) / steps
    flops = 72.0 * Nc ** 3 * V                         # 8 Nc^3 (complex Gauss-Jordan) + 8 x 8 Nc^3 (products), real flops
    bytes_alg = V * (9 + 9) * Nc * Nc * 8              # 9 matrices read, 9 written (slot 0 = identity)
    peak, peak_src = measured_peak_gbs()
    fp64_peak = 148 * 64 * 2 * 1.965e9 / 1e12          # 148 SMs x 64 DFMA lanes x 2 flop x 1.965 GHz = 37.2 TFLOP/s
    line = {
        "metric": "hat-link builds: coarse sites/s", "value": V * steps / (ms_total * steps * 1e-3), "unit": "sites/s", "n_gpus": 1,
        "steps": steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_total, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "block-preconditioned links Yhat = X^-1 Y on the %s lattice, Nc=%d, complex64 in, %s out" %
                               ("x".join(map(str, dims)), Nc, "int16 + scales" if q is not None else "complex64"),
                   "seed": cfg["seed"]},
        "clocks": clocks.summary(), "gpu_launches": (2 if q is not None else 1) * steps,
        "roofline": {"bound": "alu", "achieved": flops / (ms_build * 1e-3) / 1e12, "peak": fp64_peak, "unit": "TFLOP/s",
                     "frac": flops / (ms_build * 1e-3) / 1e12 / fp64_peak, "traffic": None,
                     "peak_source": "fp64 FMA: 148 SMs x 64 lanes x 2 flop x 1.965 GHz (derived, DESIGN.md §10)",
                     "kernel": "hat_links_kernel", "kernel_ms": ms_build, "quantize_ms": ms_total - ms_build,
                     "algorithmic_flops_per_launch": flops, "algorithmic_bytes_per_launch": bytes_alg,
                     "hbm_gbs": bytes_alg / (ms_build * 1e-3) / 1e9, "hbm_frac_of_measured": bytes_alg / (ms_build * 1e-3) / 1e9 / peak},
    }
    if parity is not None:
        line["parity"] = parity
    if not emit:
        op.close()
        return line
    print(json.dumps(line), flush=True)
    op.close()
    return 0


def run_cagcr(args, cfg, emit=True):
    """--workload cagcr: CA-GCR(8) smoother cycles on the config's operator
    (diagonally shifted so that the smoother converges).  One step = one cycle = 8 applies + 7 fused
    Chebyshev recurrence steps + the fused Gram pass + the 8x8 solve + the fused update (+ the interval estimate)."""
    import paper_2212_12559_b200 as cop
    world, rank, local = dist_env()
    if world > 1:
        raise RuntimeError("--workload cagcr is a single-GPU measurement")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dims, Nc, s = cfg["dims"], cfg["Nc"], (16 if args.cheb else 8)
    V = synth.lattice_volume(dims)
    prec = cop.LINK_I16 if cfg["links"] == "i16" else cop.LINK_C64
    links = synth.make_gamma_hermitian_links(dims, Nc, cfg["seed"], device=dev)
    links[:, 0] += 12.0 * torch.eye(Nc, dtype=torch.complex64, device=dev)

    n_launch = [0]

    def smooth(work=None):
        if args.cheb:      # caller-supplied interval: the hopping part has spectral radius ~4.1 around the shifted diagonal 12.1
            w = op.cagcr_cheb(b, x, 7.5, 16.7, s=s, cycles=1, work=work, info=info)
        else:              # the default: interval estimated on the device from the first residual
            w = op.cagcr(b, x, s=s, cycles=1, work=work, info=info)
        n_launch[0] += op.last_launches
        return w
    scales = None
    if prec == cop.LINK_I16:
        q = torch.empty((V, 9, Nc, Nc, 2), dtype=torch.int16, device=dev)
        scales = torch.empty((V, 9), dtype=torch.float32, device=dev)
        cop.coarse_op_quantize_i16(links, Nc, q, scales)
        torch.cuda.synchronize()
        links = q
    b = synth.make_vectors(dims, Nc, 1, cfg["seed"] + 1, device=dev)
    x = torch.zeros_like(b)
    op = cop.CoarseOp(dims, Nc, prec).set_links(links, scales)
    info = torch.zeros((1, 3), dtype=torch.float64, device=dev)
    work = smooth()
    stream = torch.cuda.current_stream()
    for _ in range(max(args.warmup, 3)):
        smooth(work)
    torch.cuda.synchronize()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clocks:
        n_launch[0] = 0
        t0.record(stream)
        for _ in range(args.steps):
            smooth(work)
        t1.record(stream)
        timed_launches = n_launch[0]
        tmp = torch.empty_like(b)
        a0.record(stream)
        for _ in range(args.steps):
            for _k in range(s):
                op.apply(b, tmp)
        a1.record(stream)
        torch.cuda.synchronize()
    ms_cycle = t0.elapsed_time(t1) / args.steps
    ms_applies = a0.elapsed_time(a1) / args.steps
    inf = info.cpu().numpy()[0]
    line = {
        "metric": METRIC, "value": s * V * args.steps / (t0.elapsed_time(t1) * 1e-3), "unit": UNIT, "n_gpus": 1,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_cycle, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "%s cycle on the %s lattice, Nc=%d, %s links (X shifted by 12): %d applies + "
                               "recurrence steps + Gram + solve + update per step" % ("Chebyshev-basis CA-GCR(16), given interval" if args.cheb else "CA-GCR(8), estimated interval",
                                                                   "x".join(map(str, dims)), Nc, cfg["links"], s),
                   "seed": cfg["seed"]},
        "clocks": clocks.summary(), "gpu_launches": timed_launches,
        "cagcr": {"ms_per_cycle": ms_cycle, "ms_of_s_plain_applies": ms_applies, "s": s,
                  "vector_side_share": 1.0 - ms_applies / ms_cycle,
                  "residual_reduction_one_cycle": float(np.sqrt(max(inf[1], 0.0) / inf[0])) if inf[0] > 0 else None,
                  "basis_vectors_kept": int(inf[2])},
    }
    if not emit:
        op.close()
        return line
    print(json.dumps(line), flush=True)
    op.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C2", choices=sorted(synth.CONFIGS))
    ap.add_argument("--workload", default="apply", choices=["apply", "schur", "cagcr", "hat"],
                    help="apply: the BASELINE metric (default); schur: the even/odd Schur-hat operator (row f1)")
    ap.add_argument("--dagger", default="both", choices=["0", "1", "both"])
    ap.add_argument("--path", type=int, default=0, help="COARSE_PATH_* override (0 = auto)")
    ap.add_argument("--stages", type=int, default=0, help="COARSE_OPT_STAGES override (0 = library default)")
    ap.add_argument("--grid", type=int, default=0, help="COARSE_OPT_GRID override (0 = one CTA per SM)")
    ap.add_argument("--fine", type=int, default=0, help="COARSE_OPT_FINE override (0 auto, 1 never, 2 always)")
    ap.add_argument("--keep-links", type=int, default=0, help="COARSE_OPT_KEEP_LINKS override (0 auto, 1 never, 2 always)")
    ap.add_argument("--graph", default="auto", choices=["auto", "on", "off"],
                    help="time all K steps as one CUDA graph (auto: when the links fit 2x L2)")
    ap.add_argument("--cheb", action="store_true", help="--workload cagcr: Chebyshev-basis CA-GCR(16) instead of CA-GCR(8)")
    ap.add_argument("--nrhs", type=int, default=0, help="override the config's number of right-hand sides")
    ap.add_argument("--nc", type=int, default=0, help="override the config's colour-spin size Nc (other compiled shapes)")
    ap.add_argument("--dims", default="", help="override the config's lattice, e.g. 16,16,8,12")
    ap.add_argument("--links", default="", choices=["", "c64", "i16"], help="override the config's link storage")
    ap.add_argument("--warp-items", type=int, default=0,
                    help="COARSE_OPT_WARP_ITEMS override (0 auto, 1 never, 2 always, 11/12/14: 1/2/4 warps per team)")
    ap.add_argument("--tensor-i8", type=int, default=0,
                    help="COARSE_OPT_TENSOR_I8: int16 links on the TENSOR path (0 auto = integer tensor cores, 1 = the 3xTF32 kernel)")
    ap.add_argument("--pdl", type=int, default=0, help="COARSE_OPT_PDL: programmatic dependent launch for chained applies (0 auto, 1 always, 2 never)")
    ap.add_argument("--hvec", action="store_true",
                    help="half-precision INPUT vectors (int16 + per-site norm, row f2) through coarse_op_apply_hvec")
    ap.add_argument("--hout", action="store_true",
                    help="half-precision OUTPUT beside the complex64 one (int16 + per-site norm, row f2) through coarse_op_apply_hout")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-parity", action="store_true", help="skip the in-run oracle comparison of sampled sites")
    ap.add_argument("--no-all-configs", dest="all_configs", action="store_false",
                    help="default C2 line only: do not attach the C1/C3/C4/C5 sub-records")
    ap.add_argument("--config-steps", type=int, default=20, help="applies per dagger for each sub-record")
    ap.add_argument("--cpu-seconds", type=float, default=10.0)
    args = ap.parse_args()
    cfg = synth.config(args.config)
    if args.nrhs:
        cfg["nrhs"] = args.nrhs
    if args.nc:
        cfg["Nc"] = args.nc
    if args.dims:
        cfg["dims"] = tuple(int(x) for x in args.dims.split(","))
    if args.links:
        cfg["links"] = args.links
    if args.nrhs or args.nc or args.dims or args.links:
        args.config = args.config + "*"          # not the BASELINE config any more: keyed tables do not apply
    daggers = [0, 1] if args.dagger == "both" else [int(args.dagger)]
    if args.workload == "schur":
        return run_schur(args, cfg)
    if args.workload == "cagcr":
        return run_cagcr(args, cfg)
    if args.workload == "hat":
        return run_hat(args, cfg)
    if args.impl == "reference":
        return run_reference(args, cfg, daggers)
    return run_ours(args, cfg, daggers)


if __name__ == "__main__":
    sys.exit(main())
