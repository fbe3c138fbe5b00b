#!/usr/bin/env python
"""bench.py -- throughput of the PPM hot path (pulse-profile evaluations per second).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ppm|reference]
                    [--workload C5|T|C1|C2|C3|C4] [--batch B] [--no-cpu-baseline | --cpu-baseline sample|full]
                    [--precision 0|1] [--tmap DEX]

A *step* is one pass of the whole hot path S0..S7 over one batch of B seeded
parameter vectors: ppm_evaluate -> ppm_fold_response -> ppm_loglike, everything through the C ABI of
include/ppm.h.  Default workload: B = 8 vectors of BASELINE.json configs[4] (C5; each vector is the
north-star target evaluation T: 2 spots x 256x256 cells, 128 phases x 300 energies, mixed-order
interpolation on the synthetic 35x11x67x166 table, fold to 1500 channels, Poisson ln L).
With N > 1 (torchrun, one rank per GPU) every rank takes its own B vectors of C5 -- independent
units, no data-path collective ("scaling": "weak"); the time is the max over ranks.

One JSON line is printed by rank 0.  `value` has the parameter batch resident in HBM; `e2e` runs
ppm_loglike_host (host parameter buffer in, host ln L out, copies inside the timed region).
`roofline` is for the dominant kernel k_cells: bound "alu" (FP64 pipe).  `achieved` / `frac` count the FP64
flop the kernel EXECUTES per launch (2 DFMA + DADD + DMUL thread instructions from the ncu capture of this very
workload and kernel source, paper_2510_07764_b200/ncu_captured.json; null when no capture matches) / the kernel's
own CUDA-event time measured inside the library on its launch stream; `algorithmic_*` is the same with the
86 flop per accumulated (cell, phase, energy) triple of SURVEY.md 8(d) (can exceed 1: the kernel shares the mu
contraction and the Lagrange -> monomial conversion between the energies of a pair).  `cpu_baseline` times the
CPU oracle as it stands on the same workload (rank 0, N = 1 only): one evaluation in full on all host threads when
that takes about a minute or less, else a bounded sample; single-threaded on a bounded sample (--cpu-baseline full:
both in full).

--precision 1 times the FP32-interpolation variant (tolerance 1e-4 instead of 1e-9; not the judged path), --tmap DEX the
per-cell temperature-map entry ppm_evaluate_map with a seeded smooth map of +-DEX around each spot's log T (with
--emission 1 | 3 | 4 under the strategies that are cubic in log T).

--impl reference: there is no reference implementation (the paper's code is not available); per
the task contract the reference arm is the CPU oracle, timed on the host cores on a bounded sample.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import gen  # noqa: E402

FLOP_PER_TRIPLE = 86.0          # SURVEY.md 8(d) accounting constant (FMA = 2 flop)
# nominal FP64 vector peak: 148 SMs x 4 sub-partitions x 16 DFMA lanes x 2 flop x 1.965 GHz
FP64_NOMINAL_TFLOPS = 148 * 4 * 16 * 2 * 1.965e9 / 1e12
METRIC = "pulse-profile evaluations per second"
UNIT = "evals/s"


def workload(name, batch, rank, world=1):
    """-> (conf dict with `batch` parameter vectors for this rank, description)."""
    from paper_2510_07764_b200.shard import shard_slice
    if name in ("C5", "T"):
        B = 1 if name == "T" else batch
        lo, hi = shard_slice(B * world, rank, world)              # weak scaling: B vectors of C5 per rank
        conf = gen.config_c5(n_vec=B * world)
        conf["params"] = np.ascontiguousarray(conf["params"][lo:hi])
        desc = ("BASELINE.json configs[4] (C5 batched likelihood): %d seeded prior vectors per GPU, each 2 spots x "
                "256x256 cells, 128 phases x 300 energies 0.2-12 keV, mixed-order interpolation on the synthetic "
                "35x11x67x166 table, banded fold 300 -> 1500 channels, Poisson ln L" % B)
        if name == "T":
            desc = "north-star target T = vector 0 of C5 evaluated alone; " + desc
        return conf, desc
    if name in ("I1", "I2"):
        conf = gen.config_interp_test(int(name[1]), n_cells=256, n_phase=128, n_energy=128)
        conf["params"] = np.ascontiguousarray(np.repeat(conf["params"], batch, axis=0))
        conf["steep_table"] = True
        return conf, ("interpolation test %s of Table 3 (PAPER.md:520-533): point-like spot, 256x256 cells, 128 phases x 128 "
                      "energies (Eq 50 grid), steep-limb synthetic table, batch of %d identical vectors per GPU" % (name[1], batch))
    conf = {"C1": gen.config_c1, "C2": gen.config_c2, "C3": gen.config_c3, "C4": gen.config_c4}[name]()
    conf["params"] = np.ascontiguousarray(np.repeat(conf["params"], batch, axis=0))
    idx = {"C1": 0, "C2": 1, "C3": 2, "C4": 3}[name]
    return conf, "BASELINE.json configs[%d] (%s), batch of %d identical vectors per GPU" % (idx, name, batch)


class ClockSampler:
    """nvidia-smi clock / throttle-reason samples (profiling recipe).  Started at process start (nvidia-smi needs a few
    hundred ms to deliver its first line); stop(t0, t1) keeps the samples whose timestamp falls inside the timed
    region [t0, t1] (time.time() values), or, for regions shorter than the sampling period, the nearest sample."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "20"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self, t0, t1):
        import datetime
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.05)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        rows = []
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.f:
            c = [x.strip() for x in line.split(",")]
            if len(c) < 8:
                continue
            try:
                ts = datetime.datetime.strptime(c[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                rows.append((ts, float(c[1]), float(c[2]), float(c[3]),
                             [n for n, v in zip(names, c[4:8]) if v.lower().startswith("active")]))
            except ValueError:
                continue
        self.f.close()
        os.unlink(self.f.name)
        inside = [r for r in rows if t0 <= r[0] <= t1]
        if not inside and rows:
            inside = [min(rows, key=lambda r: abs(r[0] - 0.5 * (t0 + t1)))]
        if inside:
            out.update(sm_mhz=statistics.median(r[1] for r in inside), sm_max_mhz=max(r[2] for r in inside),
                       reasons=sorted({n for r in inside for n in r[4]}), samples=len(inside),
                       power_w_max=max(r[3] for r in inside))
        return out


def _oracle_run(conf, atm, rsp, sel):
    import oracle as o
    cfg, E, p = conf["cfg"], conf["energies"], conf["params"][0]
    t0 = time.perf_counter()
    f, _ = o.evaluate(cfg, E, p, atm, phase_sel=sel)
    if rsp is not None:
        c = o.fold(f, rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"], p[5], rsp["n_channel"])
        o.loglike(c, np.ones_like(c), None, 1.0)
    return time.perf_counter() - t0


def oracle_sample(conf, n_extra=4, threads=None):
    """Time the CPU oracle, as it stands, on vector 0 of the workload: one run on 1 output phase and
    one on 1 + n_extra phases (the per-row template work is paid once per run, the shift-and-add
    scales with the phases), fold + ln L on the sampled phases; the full-evaluation time is the
    linear extrapolation to n_phase phases.  -> dict(value evals/s, seconds, cores, sample)."""
    import oracle as o
    cfg, E = conf["cfg"], conf["energies"]
    atm = o.Atmosphere(*(gen.steep_limb_atmosphere() if conf.get("steep_table") else gen.synthetic_atmosphere())) \
        if cfg["emission"] else None
    nph = cfg["n_phase"]
    n_extra = max(1, min(n_extra, nph - 1))
    sel1 = [nph // 3]
    sel2 = sel1 + [(nph // 3 + (i + 1) * nph // (n_extra + 1)) % nph for i in range(n_extra)]
    rsp = gen.synthetic_response(E) if len(E) == 300 else None
    all_threads = o.num_threads()
    if threads:
        o.set_num_threads(threads)
    try:
        d1 = _oracle_run(conf, atm, rsp, sel1)
        d2 = _oracle_run(conf, atm, rsp, sel2)
        cores = o.num_threads()
    finally:
        o.set_num_threads(all_threads)
    per_phase = max(d2 - d1, 0.0) / n_extra
    full = d1 + per_phase * (nph - 1)
    return dict(value=1.0 / full, seconds=d1 + d2, cores=cores, full_eval_s=full,
                sample="vector 0: oracle run on 1 and on %d of %d output phases (%.1f s + %.1f s), full evaluation "
                       "extrapolated linearly in phases to %.1f s" % (1 + n_extra, nph, d1, d2, full))


def oracle_full(conf, threads=None):
    """One whole evaluation of vector 0 by the CPU oracle (+ fold + ln L where the workload has a response)."""
    import oracle as o
    cfg, E = conf["cfg"], conf["energies"]
    atm = o.Atmosphere(*(gen.steep_limb_atmosphere() if conf.get("steep_table") else gen.synthetic_atmosphere())) \
        if cfg["emission"] else None
    rsp = gen.synthetic_response(E) if len(E) == 300 else None
    all_threads = o.num_threads()
    if threads:
        o.set_num_threads(threads)
    try:
        d = _oracle_run(conf, atm, rsp, None)
        cores = o.num_threads()
    finally:
        o.set_num_threads(all_threads)
    return dict(value=1.0 / d, seconds=d, cores=cores, full_eval_s=d,
                sample="vector 0 evaluated in full (%d phases x %d energies), %.1f s" % (cfg["n_phase"], len(E), d))


def cpu_baseline(conf, mode="sample"):
    """-> the bench line's cpu_baseline object.  All host threads: in full when the predicted time is <= 75 s (or
    mode == "full"), else the extrapolated sample; one thread: a sample (in full when mode == "full")."""
    first = oracle_sample(conf)
    allc = oracle_full(conf) if (mode == "full" or first["full_eval_s"] <= 75.0) else first
    one = oracle_full(conf, threads=1) if mode == "full" else oracle_sample(conf, n_extra=2, threads=1)
    return {"value": allc["value"], "unit": UNIT, "cores": allc["cores"], "kind": "oracle", "sample": allc["sample"],
            "s_per_eval": allc["full_eval_s"],
            "single_thread": {"value": one["value"], "unit": UNIT, "cores": one["cores"], "s_per_eval": one["full_eval_s"],
                              "sample": one["sample"]}}


def _code_only(text):
    """the source without comments and with white space collapsed: the hash follows the code, not its commentary"""
    import re
    text = re.sub(r"/\*.*?\*/", " ", text, flags=re.S)
    text = re.sub(r"//[^\n]*", " ", text)
    return " ".join(text.split())


def kernel_source_files(precision=0, tmap=False, domain=0):
    """the sources that define the cell kernel a bench configuration runs (shared code + that family's file)"""
    files = ["ppm_common.cuh", "ppm_cells.cuh"]
    if domain == 1:
        files.append("ppm_cells_lin.cuh")
    if tmap:
        files.append("ppm_cells_map.cuh")
    if precision == 1:
        files.append("ppm_cells32.cuh")
        if tmap:
            files.append("ppm_cells_map32.cuh")
    return files


def kernel_source_hash(precision=0, tmap=False, domain=0):
    """sha256 (first 16 hex digits) of the sources that define the cell kernel of this configuration, comments and white
    space excluded: a capture in ncu_captured.json is used only for the kernel source it was taken from."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2510_07764_b200", "csrc")
    for f in kernel_source_files(precision, tmap, domain):
        with open(os.path.join(d, f), "r") as fh:
            h.update(_code_only(fh.read()).encode())
    return h.hexdigest()[:16]


def ncu_capture_for(key, precision=0, tmap=False, domain=0):
    """Counters of the `ncu --set full` capture of the cell kernel on exactly this workload key and kernel source, or None."""
    path = os.path.join(ROOT, "paper_2510_07764_b200", "ncu_captured.json")
    try:
        with open(path) as f:
            cap = json.load(f).get("captures", {}).get(key)
    except (OSError, ValueError):
        return None
    if not cap or cap.get("source_hash") != kernel_source_hash(precision, tmap, domain):
        return None
    return cap


def run_reference(args, rank):
    """Reference arm = the CPU oracle (rank 0 only)."""
    if rank != 0:
        return
    conf, desc = workload(args.workload, args.batch, 0)
    for _ in range(args.warmup):
        oracle_sample(conf, n_extra=1)
    vals, secs, last = [], 0.0, None
    t0 = time.perf_counter()
    for _ in range(args.steps):
        last = oracle_sample(conf, n_extra=2)
        vals.append(last["value"])
        secs += last["seconds"]
    wall = time.perf_counter() - t0
    v = float(np.mean(vals))
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * wall / max(args.steps, 1), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": desc, "note": "reference arm = CPU oracle (oracle/ppm_oracle.c, direct quadrature), "
                                                  "each step a bounded sample: " + last["sample"]},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": last["cores"], "kind": "oracle",
                             "sample": last["sample"]},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ppm", choices=["ppm", "reference"])
    ap.add_argument("--workload", default="C5", choices=["C5", "T", "C1", "C2", "C3", "C4", "I1", "I2"])
    ap.add_argument("--emission", type=int, default=None, choices=[1, 2, 3, 4],
                    help="override the workload's interpolation strategy: 1 a, 4 b, 3 c, 2 d (PAPER.md:551)")
    ap.add_argument("--interp-domain", type=int, default=0, choices=[0, 1],
                    help="1: the table interpolation acts on I/T^3 instead of its logarithm (reading R13g)")
    ap.add_argument("--chain", action="store_true",
                    help="time the device-resident sampler loop (ppm_chain_run: proposal kernel -> S0-S7 -> accept -> exchange, one "
                         "CUDA-graph replay per step, --batch walkers); e2e is then the same Metropolis step driven from the host "
                         "through ppm_loglike_host")
    ap.add_argument("--phase-interp", type=int, default=0, choices=[0, 1, 3], help="order of Interp in Eq 46 (reading R11b)")
    ap.add_argument("--batch", type=int, default=8,
                    help="parameter vectors per GPU and step (C5: BASELINE.json states 1024; the default 8 gives the "
                         "per-evaluation figure in seconds instead of minutes)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-baseline", default="sample", choices=["sample", "full"],
                    help="full: time the oracle on one whole evaluation both single-threaded and on all threads")
    ap.add_argument("--tmap", type=float, default=None, metavar="DEX",
                    help="per-cell temperature maps (ppm_evaluate_map): each spot's log T modulated by +-DEX over its mesh")
    ap.add_argument("--precision", type=int, default=0, choices=[0, 1],
                    help="0: fp64 everywhere (default, the judged path); 1: fp32 interpolation + exponential")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    args.warmup = max(args.warmup, 3)
    clocks = ClockSampler(int(os.environ.get("LOCAL_RANK", "0")))

    import torch
    import paper_2510_07764_b200 as ppm
    from paper_2510_07764_b200.shard import max_over_ranks
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the PPM hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    conf, desc = workload(args.workload, args.batch, rank, world)
    if args.emission is not None and conf["cfg"]["emission"]:
        conf["cfg"] = dict(conf["cfg"], emission=args.emission)
    conf["cfg"] = dict(conf["cfg"], interp_domain=args.interp_domain if conf["cfg"]["emission"] else 0,
                       phase_interp=args.phase_interp)
    cfg, E = conf["cfg"], conf["energies"]
    B = conf["params"].shape[0]
    ctx = ppm.PPM(cfg, E, max_batch=B, device=local, precision=args.precision)
    if cfg["emission"]:
        ctx.load_atmosphere(*(gen.steep_limb_atmosphere() if conf.get("steep_table") else gen.synthetic_atmosphere()))
    rsp = gen.synthetic_response(E)
    ctx.set_response(rsp["n_channel"], rsp["first_chan"], rsp["rsp_band"], rsp["tau_ref"])
    data_h, bkg_h = gen.synthetic_counts(cfg["n_phase"], rsp["n_channel"])
    data = torch.as_tensor(data_h, device=dev)
    bkg = torch.as_tensor(bkg_h, device=dev)
    exposure = 1.0e6
    params = torch.as_tensor(conf["params"], dtype=torch.float64, device=dev).contiguous()
    params_pinned = torch.as_tensor(conf["params"], dtype=torch.float64).contiguous().pin_memory()
    flux = torch.empty((B, cfg["n_phase"], len(E)), dtype=torch.float64, device=dev)
    status = torch.empty((B,), dtype=torch.int32, device=dev)
    counts = torch.empty((B, cfg["n_phase"], rsp["n_channel"]), dtype=torch.float64, device=dev)
    ll = torch.empty((B,), dtype=torch.float64, device=dev)
    ll_host = np.empty((B,))
    st_host = np.empty((B,), dtype=np.int32)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2

    tmap = None
    if args.tmap is not None:
        tmap = torch.as_tensor(gen.smooth_temperature_map(cfg, conf["params"], args.tmap), device=dev).contiguous()

    def step():
        if tmap is not None:
            ctx.evaluate_map(params, tmap, flux, status)
        else:
            ctx.evaluate(params, flux, status)
        ctx.fold_response(flux, params, counts)
        ctx.loglike(counts, data, bkg, exposure, ll)

    chain_box = None
    if args.chain:
        P = conf["params"].shape[1]
        lo, hi, sig = np.full(P, -1e30), np.full(P, 1e30), np.zeros(P)
        for k0, (a, b_, s_) in {0: (1.0, 3.0, 0.01), 1: (8.0, 16.0, 0.05), 3: (0.0, 1.0, 0.005), 5: (0.05, 3.0, 0.01)}.items():
            lo[k0], hi[k0], sig[k0] = a, b_, s_
        for sp_ in range(cfg["n_spots"]):
            for off, (a, b_, s_) in {0: (0.1, np.pi - 0.1, 0.005), 2: (0.05, 1.0, 0.005), 3: (5.6, 6.5, 0.002)}.items():
                lo[8 + 8 * sp_ + off], hi[8 + 8 * sp_ + off], sig[8 + 8 * sp_ + off] = a, b_, s_
        chain_box = (lo, hi, sig)
        ctx.chain_create(conf["params"], lo, hi, sig, data, bkg, exposure, seed=gen.SEED0)
        host_state = {"p": conf["params"].copy(), "ll": None, "rng": np.random.default_rng(gen.SEED0)}

    def step_chain():
        ctx.chain_run(1)

    def step_chain_host():
        """the same Metropolis step driven from the host: proposals and acceptance in numpy, ln L through ppm_loglike_host"""
        lo, hi, sig = chain_box
        if host_state["ll"] is None:
            host_state["ll"] = ctx.loglike_host(host_state["p"], data, bkg, exposure)[0].copy()
        prop = host_state["p"] + sig[None, :] * host_state["rng"].standard_normal(host_state["p"].shape)
        inside = np.all((prop >= lo) & (prop <= hi) | (sig == 0), axis=1)
        prop[~inside] = host_state["p"][~inside]
        llp, _ = ctx.loglike_host(prop, data, bkg, exposure)
        acc = inside & np.isfinite(llp) & (np.log(host_state["rng"].uniform(size=len(llp))) < llp - host_state["ll"])
        host_state["p"][acc] = prop[acc]
        host_state["ll"][acc] = llp[acc]

    def step_e2e():
        if args.chain:
            return step_chain_host()
        if tmap is not None:               # no host-buffer entry for maps: device-pointer calls + explicit copies
            params.copy_(params_pinned, non_blocking=True)
            step()
            ll_host[:] = ll.cpu().numpy()
            st_host[:] = status.cpu().numpy()
        else:
            ctx.loglike_host(params_pinned.numpy(), data, bkg, exposure, ll_host, st_host)

    def sync():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    def timed(fn, k):
        """K steps, each between two CUDA events on the launch stream; L2 flushed before every step (outside its events)."""
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * k)]
        sync()
        t0 = time.perf_counter()
        for i in range(k):
            flush.zero_()
            ev[2 * i].record()
            fn()
            ev[2 * i + 1].record()
        sync()
        wall = time.perf_counter() - t0
        per = [ev[2 * i].elapsed_time(ev[2 * i + 1]) for i in range(k)]
        total = sum(per)                                  # device time of the K steps; the L2 flushes lie between them
        t = max_over_ranks([total, wall * 1e3], device=dev)
        return t[0], t[1], per

    for _ in range(args.warmup):
        step()
    sync()
    assert int(status.sum()) == 0, "workload vectors must be inside the supported domain"
    n0 = ctx.launch_count()
    ctx.profile_enable(True)
    t_begin = time.time()
    if args.chain:
        for _ in range(args.warmup):
            step_chain()
        n0 = ctx.launch_count()
    total_ms, wall_ms, per = timed(step_chain if args.chain else step, args.steps)
    clk = clocks.stop(t_begin, time.time())
    launches = ctx.launch_count() - n0
    if args.chain:                              # the captured step holds no event records: per-kernel times from eager steps
        ctx.profile_enable(True)                # (also resets the device-side unit counter the graph replays advanced)
        timed(step, args.steps)
    prof, triples = ctx.profile_read()
    ctx.profile_enable(False)
    ll_dev = ll.cpu().numpy().copy()

    # e2e: host buffers through the C ABI, copies inside the timed region
    for _ in range(2):
        step_e2e()
    e2e_total, _, _ = timed(step_e2e, args.steps)
    assert args.chain or np.array_equal(ll_host, ll_dev), "host-buffer path must reproduce the device-pointer path bit for bit"

    ms_per_step = total_ms / args.steps
    value = world * B * args.steps / (total_ms * 1e-3)
    e2e_value = world * B * args.steps / (e2e_total * 1e-3)

    if rank == 0:
        cells_ms, cells_n = prof["cells"]
        n_launch = max(cells_n, 1)
        tri_per_launch = triples / n_launch
        kern_s = cells_ms / n_launch * 1e-3
        algorithmic = FLOP_PER_TRIPLE * tri_per_launch / kern_s / 1e12
        try:
            peak_dfma = ppm.measure_fp64_peak(local) / 1e12
        except ppm.PPMError:
            peak_dfma = None
        kern_ms = {k: round(v[0] / args.steps, 4) for k, v in prof.items()}
        table = bool(cfg["emission"])
        kname = (("k_cells_map" if args.tmap is not None else "k_cells_lin" if args.interp_domain else
                  "k_cells_tab32" if args.precision else "k_cells_tab")
                 if table else "k_cells_bb")
        key = "%s:%d:p%d%s" % (args.workload, B, args.precision, "" if args.tmap is None else ":tmap%g" % args.tmap)
        if args.emission is not None or args.interp_domain or args.phase_interp == 3:
            key += ":e%s:d%d:ph%d" % (args.emission, args.interp_domain, args.phase_interp)
        cap = ncu_capture_for(key, args.precision, args.tmap is not None, args.interp_domain)
        # precision = 1 runs the per-triple work on the FP32 pipe: 128 FFMA lanes per SM, twice the FP64 figure
        peak_nominal = FP64_NOMINAL_TFLOPS * (2.0 if args.precision == 1 else 1.0)
        achieved = exec_per_unit = traffic = None
        if cap:
            # thread-level FP64 instructions of ONE launch of this workload (deterministic): 2 flop per DFMA
            flop_per_launch = 2.0 * cap["dfma"] + cap["dadd"] + cap["dmul"] + \
                              (2.0 * cap.get("ffma", 0) + cap.get("fadd", 0) + cap.get("fmul", 0) if args.precision == 1 else 0.0)
            achieved = flop_per_launch / kern_s / 1e12
            exec_per_unit = flop_per_launch / max(tri_per_launch, 1.0)
            traffic = cap.get("dram_bytes")
        roofline = {"bound": "alu", "kernel": kname,
                    "achieved": achieved, "peak": peak_nominal, "unit": "TFLOP/s",
                    "frac": (achieved / peak_nominal) if achieved is not None else None,
                    "traffic": traffic,
                    "basis": ("executed FP64 flop per launch (2 DFMA + DADD + DMUL thread instructions, ncu capture of this "
                              "workload and kernel source: %s) / the kernel's CUDA-event time" % cap.get("profile", "?"))
                             if cap else "no ncu capture matches this workload key and kernel source: see algorithmic_*",
                    "capture_key": key, "kernel_source_hash": kernel_source_hash(args.precision, args.tmap is not None, args.interp_domain),
                    "executed_flop_per_unit": exec_per_unit,
                    "algorithmic_flop_per_unit": FLOP_PER_TRIPLE, "algorithmic_achieved": algorithmic,
                    "algorithmic_frac": algorithmic / peak_nominal,
                    "peak_source": ("nominal FP32 FMA pipe: 148 SM x 128 FFMA/clk x 2 flop x 1.965 GHz" if args.precision == 1 else
                                    "nominal FP64 FMA pipe: 148 SM x 64 DFMA/clk x 2 flop x 1.965 GHz (DESIGN.md "
                                    "Roofline); MEASURED_PEAKS.json has no FP64 entry"),
                    "peak_measured_dfma_chain": peak_dfma,
                    "frac_of_measured_dfma_chain": (achieved / peak_dfma) if (peak_dfma and achieved is not None) else None,
                    # the kernel's binding resource: shared-memory wavefronts of this launch (ncu capture) / the
                    # kernel's live CUDA-event time, against 1 wavefront (128 B) per clock and SM
                    "shared_memory": ({"wavefronts_per_launch": cap.get("smem_wavefronts"),
                                       "achieved_gwavefronts_per_s": cap["smem_wavefronts"] / kern_s / 1e9,
                                       "peak_gwavefronts_per_s": 148 * 1.965,
                                       "frac": cap["smem_wavefronts"] / kern_s / (148 * 1.965e9)}
                                      if (cap and cap.get("smem_wavefronts")) else None),
                    "ncu_utilisation": ({"note": "same ncu capture; the highest of the three is the kernel's binding resource (DESIGN.md 6)",
                                         "shared_memory_wavefronts_pct_of_peak": cap.get("smem_wavefronts_pct"),
                                         "fp64_pipe_pct_of_peak": cap.get("fp64_pipe_pct"),
                                         "issue_active_pct": cap.get("issue_active_pct")} if cap else None),
                    "units_per_launch": tri_per_launch, "unit_name": "accumulated (cell, phase, energy) triple",
                    "kernel_ms_per_launch": cells_ms / n_launch, "kernel_launches_per_step": cells_n / args.steps,
                    "kernel_share_of_step": cells_ms / total_ms, "kernel_ms_per_step": kern_ms}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_per_step, "ms_per_eval": ms_per_step / B,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64" if args.precision == 0 else "f32 interpolation / f64 geometry+sums", "data": "synthetic",
                "config": {"emission": cfg["emission"], "interp_domain": cfg["interp_domain"], "phase_interp": cfg["phase_interp"],
                           "workload": desc + (" -- NOTE: BASELINE.json states a batch of 1024 for this config; this run uses "
                                               "%d per GPU (per-evaluation figure; run --batch 1024 for the stated batch)" % B
                                               if args.workload == "C5" and B != 1024 else ""), "name": args.workload, "precision": args.precision, "tmap_dex": args.tmap, "batch_per_gpu": B, "sub_batch": ctx.sub_batch(), "n_fp": ctx.n_fp,
                           "l2": "flushed before every step (256 MiB write between the steps' CUDA-event brackets)",
                           "step": ("ppm_chain_run(1): proposal kernel + S0-S7 + accept + exchange, one CUDA-graph replay, %d walkers" % B)
                                   if args.chain else "ppm_evaluate + ppm_fold_response + ppm_loglike (S0-S7)"},
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(params_pinned.numel() * 8),
                        "d2h_bytes_per_step": int(ll_host.nbytes + st_host.nbytes),
                        "call": "host-driven Metropolis step: numpy proposals + ppm_loglike_host + numpy acceptance" if args.chain
                                else "ppm_loglike_host (host params in, host ln L + status out)"},
                "gpu_launches": int(launches), "clocks": clk, "wall_ms_per_step": wall_ms / args.steps,
                "step_ms": [round(x, 3) for x in per], "roofline": roofline, "cpu_baseline": None}
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(conf, args.cpu_baseline)
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
