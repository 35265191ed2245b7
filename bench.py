#!/usr/bin/env python
"""bench.py -- throughput of the whole hot path (bz_step + bz_moments: SURVEY.md 8a rows a1-a8) on synthetic input.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..4] [--impl ours|reference] [--slab]

Default workload: BASELINE.json configs[4] (16^3 spatial x 24^3 momentum cells, 7 species, 64 samples per cell:
3.6e9 kinematic samples and 3.96e8 phase-space values per step, 3.17 GB per copy of f) -- the largest config, the one
north_star quotes the roofline target on; it fits one GPU.  One JSON line is printed by rank 0.

  value            kinematic collision samples per second over the whole step, inputs resident in HBM
  e2e              the same, but every step starts from HOST f in pinned memory and ends with f and the moments back on
                   the host (bz_step_host: copies, collision and stream + Euler pipelined by z layers; then bz_moments)
  roofline         the collision kernel alone (CUDA events inside libbz.so around every launch of the timed region).
                   north_star's roofline is the SLOWER of two legs; both are computed, the binding one is `roofline`, the
                   other `roofline_other_leg`.  HBM leg ("bound": "hbm"): ACCEPTANCE-WEIGHTED gathered/scattered bytes --
                   only samples with both outgoing legs in the box gather and scatter (reading S9), the kernel counts them
                   (bz_get_sample_counts), so bytes per generated sample = acceptance x 48 S + 16 S / N_s; its
                   `frac_survey_8d_literal` is SURVEY.md 8d's count as written (every sample credited with 3 cells x S x
                   16 B).  FP64 leg ("bound": "alu"): the operation count of the method as the oracle's source states it
                   (per generated sample, per accepted sample, per channel) against the measured FP64 peak.
  cpu_baseline     the oracle as it stands, on this box's host cores, on a bounded sample of the same workload

N > 1: bench.py starts its own ranks (torch.distributed.run, one per GPU, NCCL) unless it already runs under torchrun.
Weak scaling by domain decomposition (paper_1912_04457_b200/slab.py): the domain is the config repeated N
times along z, every rank owns one copy and exchanges one boundary layer with each z neighbour per step (the drift
stencil's only coupling); collisions are local.  The max over ranks of the device time is used.
--impl reference: the oracle arm (rank 0 only), each step a bounded sample of the workload.
"""
import argparse
import csv
import json
import os
import socket
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import workloads as wl  # noqa: E402

METRIC = "collision_samples_per_sec"
UNIT = "samples/s"

# ---- operation counts of the method, frozen from oracle/bzo.c (each fp64 + - x / sqrt = 1) --------
# gen_sample, per GENERATED sample: 3 uniforms (add, mul each) 6; p2 6; E2 6; d12 5; s 3; binning of p2 6; Marsaglia
# 11 per attempt x 4/pi attempts = 14, accepted direction 8; P 3, E 1, M 1; c 5; h 3; p3 12; p4 3; E3 2; d13 5; t 3;
# u 2; binning of p3, p4 12  (the p1 cell centre and E1 are per cell, 15 / N_s per sample)
FLOP_PER_GENERATED = 108.0
# per ACCEPTED sample: w = K/(E1 E2) 2; Table I, the 10 distinct values with shared s^2, t^2, u^2, 1/(t - m^2),
# 1/(u - m^2): 80 (20 for the pure-glue row alone); F = 1 +- f for 4 cells x S species: 4 S
# per accepted sample AND ordered channel (collide_tile's inner loop): bracket 7, x w x |M|^2 2, four deposits 4 = 13
FLOP_PER_CHANNEL = 13.0
FLOP_PER_CHANNEL_LOW = 8.0          # the lower end of SURVEY.md 8d's "8-13 flop per channel"
FP64_NOMINAL_TFLOPS = 37.2          # 148 SMs x 64 FP64 lanes x 2 x 1.965 GHz
N_CHANNELS = {1: 1, 6: 90, 7: 127}


def flop_per_accepted(cfg, per_channel=FLOP_PER_CHANNEL):
    n_ch = N_CHANNELS.get(cfg.S)
    if n_ch is None:
        return None
    return 2.0 + (20.0 if cfg.S == 1 else 80.0) + 4.0 * cfg.S + per_channel * n_ch


def negative_msq_report(g, cfg, step):
    """Reading S8: the fraction of (sample, channel) pairs whose regulated Table I value is negative, over
    the samples bz_collision draws at `step` in a bounded block of spatial cells, for the f the context holds now.  Counted
    on the device (bz_msq_sign_counts); the ordered-channel multiplicity of every (kind, ordering) is the library's table."""
    from paper_1912_04457_b200 import bz
    cells = min(cfg.Nx, 64)
    x0 = (cfg.Nx - cells) // 2
    accepted, neg = g.msq_sign_counts(step, x0, x0 + cells)
    mult = [[0, 0] for _ in range(7)]
    for row in bz.debug_paper_channels(cfg.species):
        mult[int(row[4])][int(row[5])] += 1
    n_ch = sum(a + b for a, b in mult)
    pairs = sum(mult[k][c] * neg[k][c] for k in range(7) for c in range(2))
    return {"fraction_of_sample_channel_pairs": pairs / (accepted * n_ch) if accepted else None,
            "samples_accepted": accepted, "ordered_channels": n_ch, "negative_pairs": pairs,
            "negative_samples_by_kind": {k: neg[i] for i, k in enumerate(bz.KINDS)},
            "sample": "spatial cells %d..%d of %d, every momentum cell and sample, Philox step %d" % (x0, x0 + cells - 1, cfg.Nx, step),
            "what": "regulated Table I evaluated literally, no clamp (reading S8); [straight, crossed] counts per kind"}


def bytes_literal_8d(cfg):
    """SURVEY.md 8d as written: 3 random cells x S species x (8 B gather + 8 B scatter) for EVERY sample, plus the p1
    cell once per N_s samples."""
    return 48.0 * cfg.S + 16.0 * cfg.S / cfg.samples


def bytes_acceptance_weighted(cfg, acceptance):
    """The method's own bytes: a rejected sample gathers and scatters nothing (S9)."""
    return acceptance * 48.0 * cfg.S + 16.0 * cfg.S / cfg.samples


def ncu_traffic(kernel, workload):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu capture (profiles/ncu_traffic.csv:
    kernel, workload, commit, bytes read, bytes written, source file).  Not measured in this run: returned with its source."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    try:
        with open(path) as fh:
            rows = [r for r in csv.DictReader(fh) if r["kernel"] == kernel and r["workload"] == workload]
        if not rows:
            return None, None
        r = rows[-1]
        return float(r["dram_bytes_read"]) + float(r["dram_bytes_write"]), "%s at commit %s (ncu --set full, one launch; not measured in this run)" % (r["source"], r["commit"])
    except Exception:
        return None, None


def transport_roofline(cfg, tr_ms, tr_n, peak):
    """Stream + Euler kernel (a6 + a7): phase-space cell updates per second.  `frac` is against SURVEY.md 8d's algorithmic
    24 B per update (f read, deposit read, f_new written); `frac_kernel_bytes` against what this kernel moves by design:
    also the deposit scratch re-zeroed and the cell-major copy of the new f (the next step's gather source), both padded
    to 8 slots per cell when S > 1."""
    if not tr_n or tr_ms <= 0:
        return None
    pad = 8.0 / cfg.S if cfg.S > 1 else 0.0
    kernel_bytes = 16.0 + (24.0 * pad if cfg.S > 1 else 16.0)
    rate = cfg.n_values * tr_n / (tr_ms * 1e-3)
    ach = rate * 24.0 / 1e9
    traffic, src = ncu_traffic("transport_kernel", cfg.name)
    return {"bound": "hbm", "kernel": "transport_kernel<1> (upwind stream + Euler + deposit conversion)",
            "cell_updates_per_sec": rate, "bytes_per_value": 24.0, "achieved": ach, "peak": peak, "unit": "GB/s",
            "frac": ach / peak, "kernel_bytes_per_value": kernel_bytes, "frac_kernel_bytes": rate * kernel_bytes / 1e9 / peak,
            "ms_per_launch": tr_ms / tr_n, "traffic": traffic, "traffic_source": src}


def vlasov_probe(g, cfg, dev, reps=5):
    """NEXT rank 2, outside the timed step: thermal masses (Eq. 8-9) and the central-difference drift +
    force operator of Eq. 15 on the bench workload's current f, timed with CUDA events on the context's stream."""
    import torch
    out = torch.empty(g.shape, dtype=torch.float64, device=dev)

    def timed(fn):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    from paper_1912_04457_b200 import bz
    L = bz.lib()
    ms_mass = timed(lambda: L.bz_thermal_masses(g._h, None))
    ms_vl = timed(lambda: g.vlasov(cfg.dt, out))
    n_cls = len({0 if s == 0 else 1 + (s - 1) // 2 for s in cfg.species})
    # per value: 8 B f read + 8 B dF written + the energy table written once and read once, 8 B per (cell, mass class)
    bytes_per_value = 16.0 + 16.0 * n_cls / cfg.S
    rate = cfg.n_values / (ms_vl * 1e-3)
    return {"kernels": "energy_kernel + vlasov_class_kernel (bz_vlasov), mass_kernel (bz_thermal_masses)", "bound": "hbm",
            "ms_vlasov": ms_vl, "ms_thermal_masses": ms_mass, "cell_updates_per_sec": rate, "bytes_per_value": bytes_per_value,
            "achieved": rate * bytes_per_value / 1e9, "unit": "GB/s"}


def paper_probe(g, cfg, dev, fp64_peak, reps=2):
    """NEXT rank 1, outside the timed step: the paper's own sampler (Eq. 17-21) with the thermal masses of
    Eq. 8-9, on a bounded part of the bench workload (one z layer of spatial cells) so that it takes about a second."""
    import torch
    from paper_1912_04457_b200 import bz
    out = torch.empty(g.shape, dtype=torch.float64, device=dev)
    masses = g.thermal_masses().numpy()
    nz = cfg.nx if cfg.Nx > 1 else 1
    g.set_slab(0, 0, 1)                                      # collide only the first z layer
    cells = (cfg.Nx // nz) if cfg.Nx > 1 else 1
    samples = cells * cfg.Np * cfg.samples
    g.collision_paper(cfg.dt, 0, out)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for r in range(reps):
        g.collision_paper(cfg.dt, 1 + r, out)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    # average number of roots kept per mass tuple, from the debug export on 64 grid points of spatial cell 0
    m0 = masses[0]
    cl, _ = g.debug_paper_samples(1, 0, 0, min(64, cfg.Np), (m0[0], m0[0], m0[0], m0[0]))
    roots = float(cl[..., 1].double().mean())
    g.set_slab(0, 0, nz)
    # distinct mass tuples of spatial cell 0: classes (g, u, d, s) with bit-identical masses share their roots
    rep = [min(c2 for c2 in range(c + 1) if float(m0[c2]) == float(m0[c])) for c in range(4)]
    table = bz.debug_paper_channels(cfg.species)
    n_ch = len(table)
    tuples = len({tuple(rep[(int(k) >> (2 * leg)) & 3] for leg in range(4)) for k in table[:, 6]})
    # fp64 operations per sample, counted on the oracle's source: root solve 70 per tuple; per kept root Table I 75 +
    # weight 8; per channel and kept root 13 (bracket 7, x |M|^2, 4 deposits, 1 gross)
    flop = tuples * 70.0 + roots * tuples * 83.0 + roots * n_ch * 13.0
    rate = samples / (ms * 1e-3)
    return {"kernel": "paper_queue_kernel (bz_collision_paper)", "bound": "alu", "sample": "%d of %d spatial cells" % (cells, cfg.Nx),
            "ms": ms, "samples_per_sec": rate, "mass_tuples": tuples, "roots_per_tuple": roots, "channels": n_ch,
            "flop_per_sample": flop, "achieved": rate * flop / 1e12, "peak": fp64_peak, "unit": "TFLOP/s",
            "frac": rate * flop / 1e12 / fp64_peak if fp64_peak else None}


def weighted_probe(g, cfg, dev, which, reps=2):
    """NEXT rank 3, outside the timed step: the weighted estimators on the whole bench workload --
    "is": importance-sampled t (bz_collision_is), "box": in-box CM direction (bz_collision_box).  Both run in
    collide_kernel with another sampler; the HBM leg is acceptance-weighted like the hot path's."""
    import torch
    fn = g.collision_is if which == "is" else g.collision_box
    out = torch.empty(g.shape, dtype=torch.float64, device=dev)
    fn(cfg.dt, 0, out)
    torch.cuda.synchronize()
    g.sample_counts(reset=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for r in range(reps):
        fn(cfg.dt, 1 + r, out)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    gen, acc = g.sample_counts(reset=True)
    rate = cfg.samples_per_step / (ms * 1e-3)
    acceptance = acc / gen if gen else None
    bps = bytes_acceptance_weighted(cfg, acceptance or 0.0)
    return {"kernel": "collide_kernel<mask, sampler %d> + finalize_kernel (bz_collision_%s)" % (1 if which == "is" else 2, which), "bound": "hbm",
            "ms": ms, "samples_per_sec": rate, "acceptance": acceptance, "accepted_samples_per_sec": rate * (acceptance or 0.0),
            "bytes_per_sample": bps, "achieved": rate * bps / 1e9, "unit": "GB/s",
            "bytes_per_sample_survey_8d_literal": bytes_literal_8d(cfg)}


def samples_rate(cfg, steps, ms):
    return cfg.samples_per_step * steps / (ms * 1e-3)


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks and throttle reasons during the timed region (the recipe's clocks line)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt, self.proc = index, [], threading.Event(), None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append([x.strip() for x in line.split(",")])
                if self._stop_evt.is_set():
                    break
        except Exception:
            pass

    def stop(self):
        self._stop_evt.set()
        if self.proc:
            self.proc.terminate()
        sm, mx, reasons = [], 0.0, set()
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons),
                "samples": len(sm)}


ORACLE_TILES_PER_CORE = 6        # the ONE bounded oracle sample both cpu_baseline and --impl reference time


def oracle_sample(cfg, f0, cores):
    """An oracle context holding M spatial cells of the workload (evenly spaced over the grid) as a bounded sample."""
    from oracle import bzo
    M = max(1, min(cfg.Nx, cores * ORACLE_TILES_PER_CORE if cfg.Nx > 1 else 1))
    xs = (np.arange(M) * (cfg.Nx // M)).astype(np.int64)
    o = bzo.Oracle(nx=M, ny=1, nz=1, dx=cfg.dx, np_=cfg.np_, pmin=cfg.pmin, pmax=cfg.pmax, species=cfg.species,
                   alpha_s=cfg.alpha_s, m_D=cfg.m_D, seed=cfg.seed, samples=cfg.samples, threads=cores)
    o.set_f(np.ascontiguousarray(f0[xs]))
    desc = ("%s restricted to %d of %d spatial cells (every %d-th), all %d momentum cells x %d samples, %d species; "
            "one full step (collision + stream + Euler + moments)" % (cfg.name, M, cfg.Nx, max(1, cfg.Nx // M), cfg.Np,
                                                                      cfg.samples, cfg.S))
    return o, M, desc


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = os.cpu_count() or 1
    f0 = wl.initial_f(cfg)
    o, M, desc = oracle_sample(cfg, f0, cores)
    for _ in range(args.warmup):
        o.step(cfg.dt)
        o.moments()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.step(cfg.dt)
        o.moments()
    dt = time.perf_counter() - t0
    samples = M * cfg.Np * cfg.samples * args.steps
    v = samples / dt
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "note": "CPU oracle (oracle/bzo.c), each step a bounded sample: " + desc},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": o_threads(o), "kind": "oracle", "sample": desc},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "cell_updates_per_sec": M * cfg.S * cfg.Np * args.steps / dt,
    }))


def o_threads(o):
    from oracle import bzo
    return int(bzo.lib().bzo_get_threads(o._h))


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def spawn_ranks(args):
    """python bench.py --gpus N outside torchrun: start the N ranks ourselves (one process per GPU, NCCL over NVLink)."""
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit("bench.py: --gpus %d but this box has %d CUDA device(s)" % (args.gpus, have))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")           # the communicator's init lines (ranks, transport) are what a scaling run is checked by
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    raise SystemExit(subprocess.call(cmd, env=env))


def run_ours(args, cfg):
    global bz
    import torch
    import torch.distributed as dist

    from paper_1912_04457_b200 import bz

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU path (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def make(nz):
        return bz.Boltzmann(nx=cfg.nx, ny=cfg.nx, nz=nz, dx=cfg.dx, np_=cfg.np_, pmin=cfg.pmin, pmax=cfg.pmax,
                            species=cfg.species, alpha_s=cfg.alpha_s, m_D=cfg.m_D, seed=cfg.seed, samples=cfg.samples, device=dev)

    f0 = wl.initial_f(cfg)
    slabs = cfg.Nx > 1 and (world > 1 or args.slab)     # --slab: the N > 1 code path on one GPU (halo layers from itself)
    if slabs:
        # weak scaling by domain decomposition: the global domain is the config repeated `world` times
        # along z (nx x ny x nz*world, periodic); every rank owns one copy plus two halo layers and exchanges one
        # boundary layer with each z neighbour per step (NCCL send/recv), collisions stay local
        from paper_1912_04457_b200 import slab
        dom = slab.SlabDomain(make, cfg.nx, cfg.nx, cfg.nx * world, rank, world)
        g = dom.engine
        nl = cfg.nx * cfg.nx
        f_local = np.zeros(((cfg.nx + 2) * nl, cfg.S, cfg.Np))
        f_local[nl:-nl] = f0
        host_in = torch.from_numpy(f_local).pin_memory()
        step_fn = dom.step
        own_values = cfg.n_values
    else:
        g = make(cfg.nx)
        host_in = torch.from_numpy(f0).pin_memory()
        step_fn = g.step
        own_values = cfg.n_values
    host_out = torch.empty_like(host_in).pin_memory()
    mom_host = torch.empty(2 * cfg.S * g.Nx + 2 * cfg.S + g.Nx, dtype=torch.float64).pin_memory()
    g.set_f(host_in)
    small = cfg.n_values * 8 * 3 < 256e6                    # footprint below ~2x L2: flush L2 between steps
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev) if small else None

    def one_step():
        step_fn(cfg.dt)
        g.moments(mom_host)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        one_step()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
        time.sleep(0.3)
    g.set_profile(True)
    g.get_profile(0)
    g.get_profile(1)
    g.sample_counts(reset=True)
    barrier()
    launches0 = bz.launch_count()
    ms = 0.0
    if small:
        for _ in range(args.steps):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            one_step()
            e1.record()
            torch.cuda.synchronize()
            ms += e0.elapsed_time(e1)
    else:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            one_step()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
    barrier()
    launches = bz.launch_count() - launches0
    coll_ms, coll_n = g.get_profile(0)
    tr_ms, tr_n = g.get_profile(1)
    generated, accepted = g.sample_counts(reset=True)
    g.set_profile(False)
    clocks = sampler.stop() if sampler else None          # the clocks of the timed region only, not of the probes below
    fp64_peak = bz.measure_fp64_peak() if rank == 0 else 0.0
    rank2 = vlasov_probe(g, cfg, dev) if (rank == 0 and cfg.Nx > 1 and not slabs and not args.no_probes) else None
    rank1 = paper_probe(g, cfg, dev, fp64_peak) if (rank == 0 and not slabs and not args.no_probes) else None
    rank3 = weighted_probe(g, cfg, dev, "is") if (rank == 0 and not slabs and not args.no_probes) else None
    rank3b = weighted_probe(g, cfg, dev, "box") if (rank == 0 and not slabs and not args.no_probes) else None
    N1 = float(mom_host[2 * cfg.S * g.Nx:2 * cfg.S * g.Nx + 2 * cfg.S:2].sum())
    neg_msq = negative_msq_report(g, cfg, args.warmup + args.steps) if (rank == 0 and not slabs) else None

    # ---- bz_step_n: the same steps without returning to the host in between (captured CUDA graph), moments once at the end
    stepn = None
    if rank == 0 and not slabs:
        nn = max(args.steps, 200 if small else args.steps)
        g.step_n(cfg.dt, 4)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g.step_n(cfg.dt, nn)
        g.moments(mom_host)
        e1.record()
        torch.cuda.synchronize()
        ms_n = e0.elapsed_time(e1)
        stepn = {"steps": nn, "ms_per_step": ms_n / nn, "samples_per_sec": samples_rate(cfg, nn, ms_n),
                 "what": "bz_step_n(%d) + one bz_moments: two steps per replay of a captured CUDA graph, Philox step word on the device" % nn}

    # ---- end to end: host f in, host f and moments out, every step
    e2e_steps = args.steps
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(e2e_steps):
        if slabs:
            dom.step_host(cfg.dt, host_in, host_out)   # boundary layers up, halo exchange, then bz_step_host over the own layers
        else:
            g.step_host(cfg.dt, host_in, host_out)     # bz_step_host: H2D, collision, stream + Euler, D2H pipelined by z layers
        g.moments(mom_host)
    e1.record()
    torch.cuda.synchronize()
    ms_e2e = e0.elapsed_time(e1)
    barrier()

    t = torch.tensor([ms, ms_e2e, coll_ms, tr_ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms, ms_e2e, coll_ms, tr_ms = (float(x) for x in t.cpu())
    ranks_ran = world
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    samples_step = cfg.samples_per_step
    value = world * samples_step * args.steps / (ms * 1e-3)
    e2e_value = world * samples_step * e2e_steps / (ms_e2e * 1e-3)
    peak, peak_src = measured_peaks()
    acceptance = accepted / generated if generated else None
    coll_s = coll_ms * 1e-3
    kern_rate = samples_step * coll_n / coll_s if coll_s > 0 else None
    roof = roof64 = None
    if kern_rate and acceptance is not None:
        b_aw, b_lit = bytes_acceptance_weighted(cfg, acceptance), bytes_literal_8d(cfg)
        ach = kern_rate * b_aw / 1e9
        traffic, tsrc = ncu_traffic("collide_kernel", cfg.name)
        fpa = flop_per_accepted(cfg)
        roof = {"bound": "hbm", "kernel": "collide_kernel (CUDA events inside libbz.so around every launch)",
                "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "peak_source": peak_src,
                "weighting": "acceptance-weighted: bytes per generated sample = acceptance x 48 S + 16 S / N_s (a rejected sample gathers and scatters nothing)",
                "acceptance": acceptance, "samples_generated": generated, "samples_accepted": accepted,
                "bytes_per_sample": b_aw, "samples_per_launch": samples_step, "ms_per_launch": coll_ms / coll_n,
                "bytes_per_sample_survey_8d_literal": b_lit, "frac_survey_8d_literal": kern_rate * b_lit / 1e9 / peak,
                "traffic": traffic, "traffic_unit": "bytes per launch (ncu dram read + write)", "traffic_source": tsrc}
        if fpa and fp64_peak:
            flop = FLOP_PER_GENERATED + acceptance * fpa
            a64 = kern_rate * flop / 1e12
            fpa_low = flop_per_accepted(cfg, FLOP_PER_CHANNEL_LOW)
            a64_low = kern_rate * (FLOP_PER_GENERATED + acceptance * fpa_low) / 1e12
            roof64 = {"bound": "alu", "kernel": "collide_kernel", "achieved": a64, "peak": fp64_peak, "unit": "TFLOP/s",
                      "frac": a64 / fp64_peak, "peak_source": "measured (bz_measure_fp64_peak, register-resident DFMA chains; an FMA counts 2)",
                      "kind": "ALGORITHMIC flop rate: the method's operations per sample x samples/s, not executed instructions -- a factorised kernel is credited with the channel-by-channel count and could exceed 1.0; it is north_star's FP64 leg, not a pipe utilisation",
                      "frac_nominal_peak": a64 / FP64_NOMINAL_TFLOPS, "nominal_peak": FP64_NOMINAL_TFLOPS,
                      "nominal_peak_source": "SURVEY.md 8d: 148 SMs x 64 FP64 lanes x 2 flop x 1.965 GHz",
                      "frac_at_8_flop_per_channel": a64_low / fp64_peak, "frac_nominal_peak_at_8_flop_per_channel": a64_low / FP64_NOMINAL_TFLOPS,
                      "executed": "ncu at round 2 (profiles/r2_collide_kernel_ncu_full.md): about 300 FP64 instructions per accepted sample, FP64 pipe 46.5 % busy, issue port about 95 % of what the instruction mix allows",
                      "flop_per_sample": flop, "flop_per_generated_sample": FLOP_PER_GENERATED, "flop_per_accepted_sample": fpa,
                      "flop_per_channel": FLOP_PER_CHANNEL, "channels": N_CHANNELS.get(cfg.S),
                      "count": "the method as oracle/bzo.c states it (channel by channel), each + - x / sqrt = 1; the kernel's factorised channel algebra executes fewer (DESIGN.md 6)",
                      "issue_port": "a DFMA holds B200's issue port for 2 cycles: the kernel's instruction mix runs at ~95 % of the port (profiles/r2_collide_issue_model.md)",
                      "ms_per_launch": coll_ms / coll_n,
                      "traffic": traffic, "traffic_unit": "bytes per launch (ncu dram read + write)", "traffic_source": tsrc}
            # north_star: "the slower of FP64 FMA peak and gathered/scattered bytes at HBM bandwidth" = the leg with the
            # lower bound on samples/s = the larger achieved fraction; that one is reported as `roofline`
            roof["binding_leg"] = roof64["binding_leg"] = "fp64" if roof64["frac"] > roof["frac"] else "hbm"
            for r in (roof, roof64):
                r["bound_samples_per_sec"] = kern_rate / r["frac"]
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": ranks_ran, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "spatial_cells": cfg.Nx, "momentum_cells": cfg.Np, "species": cfg.S,
                   "samples_per_cell": cfg.samples, "dt_fm": cfg.dt, "samples_per_step": samples_step,
                   "phase_space_values": cfg.n_values, "step": "bz_step + bz_moments",
                   "l2": "L2 flushed between steps (256 MB write)" if small else "inputs larger than L2 (3 x %.2f GB)" % (cfg.n_values * 8 / 1e9),
                   "parallelism": ("z slabs, one halo layer exchanged with each neighbour per step (NCCL send/recv), domain = config x %d along z" % world if slabs
                                   else "independent replicas (homogeneous config: nothing to exchange)" if world > 1 else "1 GPU")},
        "cell_updates_per_sec": world * cfg.n_values * args.steps / (ms * 1e-3),
        "samples_x_channels_per_sec": value * N_CHANNELS[cfg.S] if cfg.S in N_CHANNELS else None,     # SURVEY.md 8d "Metric" (i)
        "negative_msq": neg_msq,                                                                       # reading S8
        "collision_kernel_samples_per_sec": kern_rate,
        "collision_kernel_accepted_samples_per_sec": kern_rate * acceptance if (kern_rate and acceptance is not None) else None,
        "collision_kernel_share_of_step": coll_ms / ms if ms > 0 else None,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": own_values * 8,
                "d2h_bytes_per_step": own_values * 8 + mom_host.numel() * 8, "ms_per_step": ms_e2e / e2e_steps},
        "gpu_launches": launches,
        "step_n": stepn,
        "roofline": roof64 if (roof64 and roof64["frac"] > roof["frac"]) else roof,
        "roofline_other_leg": roof if (roof64 and roof64["frac"] > roof["frac"]) else roof64,
        "roofline_transport": transport_roofline(cfg, tr_ms, tr_n, peak),
        "next_rank1_paper_sampler": rank1,
        "next_rank3_importance_sampling": None if rank3 is None else dict(rank3, peak=peak, frac=rank3["achieved"] / peak),
        "next_rank3_inbox_sampling": None if rank3b is None else dict(rank3b, peak=peak, frac=rank3b["achieved"] / peak),
        "next_rank2_eq15": None if rank2 is None else dict(rank2, peak=peak, frac=rank2["achieved"] / peak),
        "clocks": clocks,
        "total_particle_number": N1,
    }
    if world == 1 and not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        o, M, desc = oracle_sample(cfg, f0, cores)
        t0 = time.perf_counter()
        o.step(cfg.dt)
        o.moments()
        dt = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": M * cfg.Np * cfg.samples / dt, "unit": UNIT, "cores": o_threads(o), "kind": "oracle",
                               "sample": desc, "seconds": dt}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-probes", action="store_true", help="skip the NEXT-row probes that run after the timed steps (for profiling the step alone)")
    ap.add_argument("--slab", action="store_true", help="run the slab-decomposition path (the N > 1 path) even on one GPU")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    cfg = wl.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args)
    run_ours(args, cfg)


if __name__ == "__main__":
    main()
