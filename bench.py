#!/usr/bin/env python
"""bench.py -- TSM sources/sec at 32^3x64 (BASELINE.json metric) on B200, with the kernel rooflines.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference] [--config c1|c3|c4]
                    [--scaling strong|weak] [--what step|dslash|dslash_group|contract|blas|solve]

One "step" = one pass of the whole hot path over one batch of synthetic input: the full TSM
estimator loop of BASELINE.json config c4 (N_LP = 500 Z4 sources solved with 16-bit storage to
rho = 1e-2, N_HP = 20 of them solved mixed fp32/fp64 to rho = 1e-8, every solution contracted into
the 160 insertions and projected onto the 123 momenta with p^2 <= 9 for all 64 timeslices).
`value` = N_LP sources / step time, inputs (gauge field, packed Z4 noise) resident in HBM.
`e2e` = the same through the host-buffer entry point: gauge field and packed noise start in pinned
host memory, the estimate ends in pinned host memory, all copies inside the timed region.
N > 1 (torchrun): the sources of the ONE (N_LP, N_HP) workload are sharded round-robin over the
ranks (strong scaling; `--scaling weak` runs N times the workload instead), the only exchange is one
all-reduce of the three raw 20 MB accumulators per step (paper_1401_6750_b200/multi.py).

`--what X` (X != step) runs one kernel family a few times on the c4 fields and prints CUDA-event
timings: the command every ncu capture under profiles/ wraps (`<cmd> && ncu ... <cmd>`).

`--impl reference` times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the
same workload on the host cores; see cpu_baseline in the JSON line.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import re
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1401_6750_b200 import inputs  # noqa: E402

LP = dict(sloppy="f16", outer="f32", recon=12, rho=1e-2, max_iter=2000, delta=0.01)
HP = dict(sloppy="f32", outer="f64", recon=12, rho=1e-8, max_iter=5000, delta=1e-4)     # delta: see DESIGN.md sec 10
GROUP = 8                       # sources per launch inside tsm_estimate (TM_OPT_GROUP automatic at c4)
PREC_BYTES = {"f64": 8, "f32": 4, "f16": 2, "bf16": 2}

# Algorithmic work of the fused contraction + projection per lattice site:
#   bytes (fp32): s and eta once (2 x 24 reals) + the 4 forward links in reconstruct-12 (4 x 12 reals)
#   flop: 16 SU(3) x spinor products (36 complex MACs each), 10 colour-traced outer products (48 complex MACs each),
#         the x-stage of the separable DFT (320 reals x 7 weights, 13 flop per real); a complex MAC = 8 flop
CONTRACT_BYTES_PER_SITE = (2 * 24 + 4 * 12) * 4
CONTRACT_FLOP_PER_SITE = 16 * 36 * 8 + 10 * 48 * 8 + 320 * 13


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def source_sha(*names):
    h = hashlib.sha256()
    for n in names:
        with open(os.path.join(ROOT, "paper_1401_6750_b200", "csrc", n), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_traffic(profile, *sources):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` summary
    profiles/<profile>, or (None, why) when there is none or when it was captured from other kernel sources than the
    ones in the tree (the summary carries the sha256 of the .cu files it was taken from)."""
    p = os.path.join(ROOT, "profiles", profile)
    if not os.path.exists(p):
        return None, "no capture committed"
    text = open(p).read()
    m = re.search(r"kernel-source-sha256: ([0-9a-f]+)", text)
    if not m or m.group(1) != source_sha(*sources):
        return None, "profiles/%s is stale (captured from another version of %s)" % (profile, "+".join(sources))
    tot, scale = 0.0, {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    for m in re.finditer(r"`dram__bytes_(?:read|write)\.sum` \| ([0-9.,]+) \| (\w+)", text):
        tot += float(m.group(1).replace(",", "")) * scale[m.group(2)]
    return (tot or None), "profiles/" + profile


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,power.draw,power.limit")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, pl, reasons = [], [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except Exception:
                continue
            for n, v in zip(names, r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
            try:
                pw.append(float(r[6]))
                pl.append(float(r[7]))
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm),
                "power_w": float(np.median(pw)) if pw else None, "power_limit_w": max(pl) if pl else None}


# ----------------------------------------------------------------------------- CPU oracle legs
_U_CACHE = {}


def oracle_gauge(cfg):
    key = (cfg["dims"], cfg["eps"], cfg["seed"])
    if key not in _U_CACHE:
        import torch
        from paper_1401_6750_b200 import inputs_torch
        dev = "cuda" if torch.cuda.is_available() else "cpu"
        _U_CACHE[key] = inputs_torch.gauge_field(cfg["dims"], cfg["eps"], cfg["seed"], dev).cpu().numpy()
    return _U_CACHE[key]


def cores_used():
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count()


def oracle_sample(cfg, hp=False, n_timeslices=1):
    """Bounded sample of the workload on the host cores with the oracle AS IT STANDS: one LP solve (rho = 1e-2, fp64
    CGNR on the full lattice), optionally one HP solve (rho = 1e-8), and the contraction + projection of n_timeslices
    of the T timeslices."""
    import oracle  # test infrastructure; allowed in bench.py's cpu_baseline / --impl reference legs only
    oracle.build()
    dims = cfg["dims"]
    U = oracle_gauge(cfg)
    eta = inputs.z4_source(dims, cfg["src_seed"], 0)
    mom = inputs.momentum_list(cfg.get("p2max", 9))
    t0 = time.perf_counter()
    s, iters, tr, st = oracle.solve(eta, U, cfg["kappa"], cfg["mu"], LP["rho"])
    t1 = time.perf_counter()
    oracle.loops_project(s, eta, U, cfg["kappa"], cfg["mu"], mom, -1, 0, n_timeslices)
    t2 = time.perf_counter()
    out = dict(lp_s=t1 - t0, lp_iters=iters, contract_s_per_timeslice=(t2 - t1) / n_timeslices)
    if hp:
        t3 = time.perf_counter()
        _, it_hp, _, _ = oracle.solve(eta, U, cfg["kappa"], cfg["mu"], HP["rho"])
        out.update(hp_s=time.perf_counter() - t3, hp_iters=it_hp)
    return out


def oracle_rate(cfg, smp, hp_s):
    """sources/s of the whole TSM step extrapolated from the sample: N_LP LP solves + N_HP HP solves + (N_LP + N_HP)
    contractions of T timeslices (hp_s = None: HP corrections left out)."""
    T = cfg["dims"][3]
    n_lp, n_hp = cfg["n_lp"], cfg["n_hp"]
    ct = smp["contract_s_per_timeslice"] * T
    total = n_lp * (smp["lp_s"] + ct)
    if hp_s is not None:
        total += n_hp * (hp_s + ct)
    return n_lp / total


def oracle_extras(cfg):
    """What BASELINE.md sec 3 promised beside the sampled rate: a single-thread operator application at the bench
    lattice and a COMPLETE oracle TSM run at c1 (every solve, every contraction, the combiner)."""
    import ctypes
    import oracle
    U = oracle_gauge(cfg)
    psi = inputs.z4_source(cfg["dims"], cfg["src_seed"], 1)
    ex = {}
    try:
        gomp = ctypes.CDLL("libgomp.so.1")
        nthr = cores_used()
        gomp.omp_set_num_threads(1)
        t0 = time.perf_counter()
        oracle.apply_M(psi, U, cfg["kappa"], cfg["mu"], -1)
        ex["apply_M_1thread_s"] = time.perf_counter() - t0
        gomp.omp_set_num_threads(nthr)
        t0 = time.perf_counter()
        oracle.apply_M(psi, U, cfg["kappa"], cfg["mu"], -1)
        ex["apply_M_all_cores_s"] = time.perf_counter() - t0
        # full operator = 2 parity Dslash; 1416 flop per output site of a parity Dslash with XPAY epilogue
        ex["apply_M_1thread_GFLOPs"] = 2 * 1416.0 * (inputs.volume(cfg["dims"]) // 2) / ex["apply_M_1thread_s"] / 1e9
    except OSError:
        pass
    c1 = dict(inputs.CONFIGS["c1"])
    n_lp, n_hp = 8, 2
    U1 = inputs.gauge_field(c1["dims"], c1["eps"], c1["seed"])
    mom = inputs.momentum_list(2)
    t0 = time.perf_counter()
    lp, hp = [], []
    for r in range(n_lp):
        eta = inputs.z4_source(c1["dims"], c1["src_seed"], r)
        s, _, _, _ = oracle.solve(eta, U1, c1["kappa"], c1["mu"], LP["rho"])
        lp.append(oracle.loops_project(s, eta, U1, c1["kappa"], c1["mu"], mom, -1))
        if r < n_hp:
            s, _, _, _ = oracle.solve(eta, U1, c1["kappa"], c1["mu"], HP["rho"])
            hp.append(oracle.loops_project(s, eta, U1, c1["kappa"], c1["mu"], mom, -1))
    oracle.tsm_combine(np.stack(lp), np.stack(hp))
    dt = time.perf_counter() - t0
    ex["c1_full_run"] = {"dims": list(c1["dims"]), "n_lp": n_lp, "n_hp": n_hp, "n_momenta": len(mom), "seconds": dt,
                         "sources_per_s": n_lp / dt}
    return ex


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # the HP solve is timed once (it alone is ~4x an LP solve); every step re-times the LP solve + 1/T contraction
    first = oracle_sample(cfg, hp=True)
    rates, last = [], first
    for i in range(args.warmup + args.steps):
        last = oracle_sample(cfg)
        if i >= args.warmup:
            rates.append(oracle_rate(cfg, last, first["hp_s"]))
    val = float(np.mean(rates)) if rates else oracle_rate(cfg, last, first["hp_s"])
    sample = ("per step: 1 of %d LP sources (oracle fp64 CGNR to rho=1e-2, %d iterations, %.1f s) + contraction/projection "
              "of 1 of %d timeslices (%.2f s); the HP solve (rho=1e-8, %d iterations, %.1f s) timed once before the steps; "
              "extrapolated to %d LP + %d HP solves and %d contractions"
              % (cfg["n_lp"], last["lp_iters"], last["lp_s"], cfg["dims"][3], last["contract_s_per_timeslice"],
                 first["hp_iters"], first["hp_s"], cfg["n_lp"], cfg["n_hp"], cfg["n_lp"] + cfg["n_hp"]))
    line = {"impl": "reference", "metric": "tsm_sources_per_sec", "value": val, "unit": "sources/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": cfg["n_lp"] / val * 1e3,
            "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(cfg, args),
            "cpu_baseline": {"value": val, "unit": "sources/s", "cores": cores_used(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "sources/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(cfg, args):
    lx, ly, lz, lt = cfg["dims"]
    return {"workload": "BASELINE.json configs[3] (paper-scale TSM) %dx%dx%dx%d" % (lx, ly, lz, lt) if args.config == "c4"
            else "config %s %dx%dx%dx%d" % (args.config, lx, ly, lz, lt),
            "n_lp": cfg["n_lp"], "n_hp": cfg["n_hp"], "rho_lp": LP["rho"], "rho_hp": HP["rho"],
            "lp_storage": LP["sloppy"], "hp": "f32 sloppy + f64 reliable updates", "recon": 12,
            "insertions": 160, "n_momenta": len(inputs.momentum_list(cfg["p2max"])), "kappa": cfg["kappa"], "mu": cfg["mu"],
            "gauge": "SU(3)-projected exp(i*eps*H), eps=%g, seed=%d" % (cfg["eps"], cfg["seed"]),
            "sources_counted": "N_LP per step (whole job)",
            "l2": "working set (gauge 201 MB 16-bit / 403 MB fp32 + 8 sources x 50 MB vectors per kernel) exceeds the "
                  "126 MB L2; kernel microbenchmarks rotate over 3-4 field sets",
            "parallelism": "sources of one (N_LP, N_HP) workload sharded round-robin over the ranks, one all-reduce of "
                           "the three raw accumulators per step" if args.scaling == "strong" else
                           "every rank runs the (N_LP, N_HP) workload on its own sources (N x the work), one all-reduce "
                           "of the three raw accumulators per step"}


# ----------------------------------------------------------------------------- CUDA arm: kernel microbenchmarks
def _tdt(torch, prec):
    return {"f64": torch.float64, "f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}[prec]


def _fill(torch, bufs, prec, dev, seed):
    # a device-side uniform fill in storage precision (Dslash cost is data-independent)
    g = torch.Generator(device=dev)
    g.manual_seed(seed)
    for b in bufs:
        v = b.view(_tdt(torch, prec))
        v.copy_((torch.rand(v.shape, generator=g, device=dev, dtype=torch.float32) - 0.5).to(v.dtype))


def _timed(torch, fn, n, warm):
    for i in range(warm):
        fn(i)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(n):
        fn(i)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / n


def time_dslash(ctx, tmod, torch, prec, recon, kappa, mu, napp, nb=1, op_name="XPAY"):
    """Average CUDA-event time (ms) of one parity-Dslash launch covering nb sources (nb > 1: tm_dslash_multi, the
    launch shape of the TSM loop).  in, out AND the XPAY operand rotate over 4 buffer sets (> L2 in total)."""
    P = tmod.PREC[prec]
    pb = ctx.tm_field_bytes(P, False)
    nset = 4
    mk = lambda: torch.empty(nb * pb, dtype=torch.uint8, device=ctx.tdev)
    ins, outs, xs = [mk() for _ in range(nset)], [mk() for _ in range(nset)], [mk() for _ in range(nset)]
    _fill(torch, ins + xs, prec, ctx.tdev, 1234)
    op = getattr(tmod, "TM_OP_" + op_name)

    def launch(i):
        j = i % nset
        if nb == 1:
            ctx.tm_dslash(outs[j], ins[j], xs[j], op, 0, False, kappa, mu, P, recon)
        else:
            ctx.tm_dslash_multi(outs[j], ins[j], xs[j], nb, op, 0, False, kappa, mu, P)
    return _timed(torch, launch, napp, 8)


def dslash_bytes_per_site(prec, recon, xpay):
    return (48 + 8 * recon + (24 if xpay else 0)) * PREC_BYTES[prec]     # 1 spinor in, 8 links, 1 out (+ x)


def time_contract(ctx, tmod, torch, inputs_torch, cfg, acc, ncall):
    """Average CUDA-event time (ms) of one contraction + projection as the TSM loop runs it (internal-layout fields)."""
    dims = cfg["dims"]
    mom = inputs.momentum_list(cfg["p2max"])
    P = tmod.PREC[acc]
    sets = []
    for j in range(2):      # 2 x (s, eta) x 201 MB (fp32) > L2
        s = ctx.tm_field_import(inputs_torch.z4_source(dims, 11, 2 * j, ctx.tdev), P)
        e = ctx.tm_field_import(inputs_torch.z4_source(dims, 11, 2 * j + 1, ctx.tdev), P)
        sets.append((s, e))
    out = torch.empty((2, 80, len(mom), dims[3]), dtype=torch.complex128, device=ctx.tdev)
    return _timed(torch, lambda i: ctx.loop_contract_project_fields(sets[i % 2][0], sets[i % 2][1], cfg["kappa"], cfg["mu"],
                                                                     mom, P, out), ncall, 2)


def c5_sweep(tmod, torch, inputs_torch, local, peak):
    """BASELINE.json configs[4] (bandwidth sweep, 48^3x96): standalone parity Dslash (XPAY epilogue) and the CG iteration
    rate per storage precision x reconstruct.  The 16-bit parity spinor is 255 MB here (> 126 MB L2)."""
    c5 = inputs.CONFIGS["c5"]
    dims = c5["dims"]
    dev = torch.device("cuda", local)
    U = inputs_torch.gauge_field(dims, c5["eps"], c5["seed"], dev)
    ctx = tmod.TmContext(dims, -1, local)
    ctx.tm_load_gauge(U)
    del U
    Vh = inputs.volume(dims) // 2
    eta = inputs_torch.z4_source(dims, c5["src_seed"], 0, dev)
    rows = {}
    for prec in ("f64", "f32", "f16", "bf16"):
        for recon in (12, 18):
            ms = time_dslash(ctx, tmod, torch, prec, recon, c5["kappa"], c5["mu"], 100)
            gbs = dslash_bytes_per_site(prec, recon, True) * Vh / (ms * 1e-3) / 1e9
            # CG: a fixed number of iterations (rho unreachable, max_iter = 40) so that the rate is per iteration
            outer = "f32" if prec in ("f16", "bf16") else prec
            info = None
            for _ in range(2):
                _, info = ctx.tm_cg_solve(eta, c5["kappa"], c5["mu"], prec, outer, recon, 1e-30, 40, 1e-30, raise_on_noconv=False)
            rows["%s_r%d" % (prec, recon)] = {
                "us_per_dslash": ms * 1e3, "GBps": gbs, "frac_of_hbm_peak": gbs / peak,
                "GFLOPs": 1416.0 * Vh / (ms * 1e-3) / 1e9,
                "cg_iters_per_sec": 1e3 * max(1, info["iters"]) / info["ms"]}
    ctx.close()
    return {"lattice": "48x48x48x96 (BASELINE.json configs[4])", "bytes_per_site": "(48 + 8 R + 24) x bytes per real",
            "flop_per_site": 1416, "launches_per_row": 100, "cg": "40 iterations of the even-odd CGLS solver, 16-bit rows "
            "with fp32 outer precision", "rows": rows}


def profile_mode(args, cfg):
    """--what X: run one kernel family a few times on the bench fields (for `<cmd> && ncu ... <cmd>`)."""
    import torch
    import paper_1401_6750_b200 as tmod
    from paper_1401_6750_b200 import inputs_torch
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    dims, kappa, mu = cfg["dims"], cfg["kappa"], cfg["mu"]
    U = inputs_torch.gauge_field(dims, cfg["eps"], cfg["seed"], dev)
    ctx = tmod.TmContext(dims, -1, 0)
    ctx.tm_load_gauge(U)
    del U
    Vh = inputs.volume(dims) // 2
    if args.what in ("dslash", "dslash_group"):
        nb = GROUP if args.what == "dslash_group" else 1
        if nb > 1 and args.recon != 12:
            raise SystemExit("bench.py --what dslash_group: tm_dslash_multi (the solver's grouped launch) is reconstruct-12 only")
        ms = time_dslash(ctx, tmod, torch, args.prec, args.recon, kappa, mu, args.napp, nb)
        nbytes = (nb * (48 + 24) + 8 * args.recon) * PREC_BYTES[args.prec] * Vh
        print("dslash %s r%d XPAY, %d source(s) per launch: %.1f us/launch, %.0f GB/s (spinors per source, links once per launch)"
              % (args.prec, args.recon, nb, ms * 1e3, nbytes / ms / 1e6))
    elif args.what == "contract":
        ctx.tm_set_option(tmod.TM_OPT_CONTRACT_PATH, args.contract_path)
        ms = time_contract(ctx, tmod, torch, inputs_torch, cfg, args.prec, args.napp)
        print("contract %s path %d: %.3f ms/call (xy + zsum + assemble, internal-layout inputs)" % (args.prec, args.contract_path, ms))
    elif args.what in ("solve", "blas"):
        eta = inputs_torch.z4_source(dims, cfg["src_seed"], 0, dev)
        P = LP if args.prec in ("f16", "bf16") else HP
        P = dict(P, sloppy=args.prec) if args.prec in ("f16", "bf16") else P
        info = None
        for _ in range(2):
            _, info = ctx.tm_cg_solve(eta, kappa, mu, **P)
        print("solve %s/%s rho=%g: %s" % (P["sloppy"], P["outer"], P["rho"], info))
    ctx.close()


# ----------------------------------------------------------------------------- CUDA arm: the TSM step
def run_b200(args, cfg):
    import torch
    import torch.distributed as dist
    import paper_1401_6750_b200 as tmod
    from paper_1401_6750_b200 import inputs_torch, multi

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    dims = cfg["dims"]
    V = inputs.volume(dims)
    kappa, mu = cfg["kappa"], cfg["mu"]
    mom = inputs.momentum_list(cfg["p2max"])
    # the job: strong = the BASELINE workload itself, weak = world x the workload; either way sharded round-robin
    n_lp_job = cfg["n_lp"] * (world if args.scaling == "weak" else 1)
    n_hp_job = cfg["n_hp"] * (world if args.scaling == "weak" else 1)
    n_lp, n_hp, first, stride = multi.shard(n_lp_job, n_hp_job, rank, world)
    seed = cfg["src_seed"]

    U = inputs_torch.gauge_field(dims, cfg["eps"], cfg["seed"], dev)
    z4_dev = torch.empty((n_lp, 3 * V), dtype=torch.uint8, device=dev)
    for j in range(n_lp):
        z4_dev[j] = inputs_torch.z4_packed(dims, seed, first + j * stride, dev)
    ctx = tmod.TmContext(dims, -1, local)
    ctx.tm_load_gauge(U)
    ctx.tm_set_option(tmod.TM_OPT_CONTRACT_PATH, args.contract_path)

    def step():
        return multi.tsm_estimate_sharded(ctx, n_lp_job, n_hp_job, kappa, mu, mom, LP, HP, tmod.TM_F32, tmod.TM_F64,
                                          seed=seed, z4=z4_dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    l0 = ctx.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    infos = []
    for _ in range(args.steps):
        _, info = step()
        infos.append(info)
    e1.record()
    barrier()
    clocks = sampler.stop()
    launches = ctx.launch_count() - l0
    ms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ms_per_step = float(ms.item()) / args.steps
    value = n_lp_job / (ms_per_step * 1e-3)

    # Where the step goes.  On one lane (the automatic choice when sources are solved 8 per launch) the phases of a step
    # follow one another on one stream and their event times add up to the step, so the breakdown comes from the timed
    # steps themselves; a run that used two lanes (overlapping phase times) gets one more, untimed, step on one lane.
    breakdown = None
    if not args.step_only:
        if all(i["lanes"] == 1 for i in infos):
            binfo = {k: float(np.mean([i[k] for i in infos])) for k in ("ms_total", "ms_lp_solve", "ms_hp_solve", "ms_contract")}
            src = "mean over the timed steps (one lane)"
        else:
            ctx.tm_set_option(tmod.TM_OPT_LANES, 1)
            _, binfo = step()
            torch.cuda.synchronize()
            ctx.tm_set_option(tmod.TM_OPT_LANES, 0)
            src = "one more, untimed, step on one lane (the timed steps ran two lanes, whose phase times overlap)"
        breakdown = {"lanes": 1, "ms_step": binfo["ms_total"], "ms_lp_solves": binfo["ms_lp_solve"],
                     "ms_hp_solves": binfo["ms_hp_solve"], "ms_contraction_noise_accumulate": binfo["ms_contract"],
                     "source": src}

    if args.step_only:
        # the launch-list capture under profiles/ wraps this mode: warm-up + timed steps, nothing else
        if rank == 0:
            print(json.dumps({"metric": "tsm_sources_per_sec", "value": value, "unit": "sources/s", "n_gpus": world,
                              "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "step_only": True,
                              "config": workload_config(cfg, args), "clocks": clocks, "gpu_launches": int(launches),
                              "extras": {k: float(np.mean([i[k] for i in infos])) for k in ("ms_lp_solve", "ms_hp_solve", "ms_contract")}}))
        ctx.close()
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- end to end through host buffers (pinned): gauge + noise H2D, estimate D2H, every step
    U_host = torch.empty(U.shape, dtype=U.dtype).pin_memory()
    U_host.copy_(U)
    z4_host = torch.empty(z4_dev.shape, dtype=torch.uint8).pin_memory()
    z4_host.copy_(z4_dev)
    del z4_dev
    shape = (2, 80, len(mom), dims[3])
    sums_host = torch.empty((3,) + shape, dtype=torch.complex128).pin_memory()
    out_host = torch.empty(shape, dtype=torch.complex128).pin_memory()

    def e2e_step(host_noise=True):
        ctx.tm_load_gauge_host(U_host)
        if world == 1:
            ctx.tsm_estimate_host(n_lp, n_hp, kappa, mu, mom, LP, HP, tmod.TM_F32, tmod.TM_F64,
                                  z4_host=z4_host if host_noise else None, seed=seed, out_host=out_host)
        else:
            ctx.tsm_estimate_host(n_lp, n_hp, kappa, mu, mom, LP, HP, tmod.TM_F32, tmod.TM_F64,
                                  z4_host=z4_host if host_noise else None, seed=seed, out_host=sums_host,
                                  src_first=first, src_stride=stride, partial_sums=True)
            sums = multi.allreduce_sums(sums_host.to(dev, non_blocking=True))
            out_host.copy_(ctx.tsm_combine_sums(sums, n_lp_job, n_hp_job))
        return out_host

    def time_e2e(host_noise, nstep):
        e2e_step(host_noise)
        barrier()
        w0 = time.perf_counter()
        for _ in range(nstep):
            e2e_step(host_noise)
        barrier()
        t = torch.tensor([(time.perf_counter() - w0) / nstep], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    e2e_s = time_e2e(True, args.steps)
    e2e_dev_noise_s = time_e2e(False, max(1, min(args.steps, 3)))
    e2e = {"value": n_lp_job / e2e_s, "unit": "sources/s",
           "h2d_bytes_per_step": int(U_host.numel() * 16 + z4_host.numel()),
           "d2h_bytes_per_step": int((sums_host if world > 1 else out_host).numel() * 16), "steps": args.steps,
           "timing": "host wall clock around the synchronous host-buffer call (gauge upload + pack, noise upload per "
                     "group on a copy stream, estimate download), max over ranks",
           "with_device_generated_noise": {"value": n_lp_job / e2e_dev_noise_s, "unit": "sources/s",
                                           "h2d_bytes_per_step": int(U_host.numel() * 16),
                                           "note": "Z4 noise from the counter hash on the device (row f1): only the gauge "
                                                   "field crosses PCIe"}}
    del U_host, z4_host

    if rank != 0:
        ctx.close()
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- rooflines, measured live with CUDA events
    peak, peak_src = peaks()
    Vh = V // 2
    napp = 200
    ds = {}
    for prec, recon in (("f16", 12), ("bf16", 12), ("f16", 18), ("bf16", 18), ("f32", 12), ("f64", 12)):
        t_ms = time_dslash(ctx, tmod, torch, prec, recon, kappa, mu, napp)
        nbytes = dslash_bytes_per_site(prec, recon, True) * Vh
        ds[prec + "_r%d" % recon] = {"us": t_ms * 1e3, "GBps": nbytes / (t_ms * 1e-3) / 1e9, "frac_of_hbm_peak": nbytes / (t_ms * 1e-3) / 1e9 / peak,
                                     "GFLOPs": 1416.0 * Vh / (t_ms * 1e-3) / 1e9}
    # the dominant kernel IN THE LAUNCH SHAPE THE TIMED STEP USES: GROUP sources per launch, links read from HBM once per
    # group (later readers hit L2).  Algorithmic bytes of such a launch: spinors per source, links once.
    sl = LP["sloppy"]
    t_g = time_dslash(ctx, tmod, torch, sl, 12, kappa, mu, 60, GROUP)
    must_move = (GROUP * (48 + 24) + 8 * 12) * PREC_BYTES[sl] * Vh
    traffic, traffic_src = ncu_traffic("r02_dslash16_f16_group8.md", "dslash.cu")
    single = ds[sl + "_r12"]
    traffic1, traffic1_src = ncu_traffic("r02_dslash16_f16.md", "dslash.cu")
    roofline = {
        "bound": "hbm", "kernel": "%s<%s> reconstruct-12 XPAY (second half of Mhat), %d sources per launch "
                                  "(the launch shape of the timed step)"
                                  % ("dslash16_group_kernel" if sl == "f16" else "dslash16_kernel", sl, GROUP),
        "achieved": must_move / (t_g * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
        "frac": must_move / (t_g * 1e-3) / 1e9 / peak, "traffic": traffic, "traffic_source": traffic_src,
        "peak_source": peak_src, "algorithmic_bytes_per_launch": must_move,
        "us_per_launch": t_g * 1e3, "us_per_source": t_g * 1e3 / GROUP,
        "how": "CUDA events around 60 back-to-back launches on the current stream, 4 rotating buffer sets of 8 sources",
        "note": "one CTA per 128 sites does the 8 sources one after the other (links staged and rebuilt once), so the "
                "launch moves 0.5x the bytes of 8 single-source launches and is bound by instruction issue and board power, "
                "not by HBM (DESIGN.md sec 6); per source it is faster than the single-source launch below",
        "single_source_equivalent_GBps": GROUP * dslash_bytes_per_site(sl, 12, True) * Vh / (t_g * 1e-3) / 1e9,
        "single_source_launch": {"us": single["us"], "achieved": single["GBps"], "frac": single["GBps"] / peak,
                                 "algorithmic_bytes_per_launch": dslash_bytes_per_site(sl, 12, True) * Vh,
                                 "traffic": traffic1, "traffic_source": traffic1_src,
                                 "how": "CUDA events around %d back-to-back launches, 4 rotating buffer sets" % napp}}

    # the contraction + projection: co-limited by the fp32 pipe, not by HBM -> both fractions, against MEASURED peaks
    fma_peak = max(ctx.tm_fma_peak(1, 8192), ctx.tm_fma_peak(0, 8192))
    t_c = time_contract(ctx, tmod, torch, inputs_torch, cfg, "f32", 20)
    t_c64 = time_contract(ctx, tmod, torch, inputs_torch, cfg, "f64", 4)
    cbytes, cflop = CONTRACT_BYTES_PER_SITE * V, CONTRACT_FLOP_PER_SITE * V
    ctraffic, ctraffic_src = ncu_traffic("r02_contract_f32.md", "contract_tma.cu", "contract.cuh")
    roofline_contract = {
        "bound": "alu", "kernel": "loop_contract_project (fp32): site stage + x/y DFT + z-sum + assembly, one source",
        "ms_per_source": t_c, "achieved": cflop / (t_c * 1e-3) / 1e12, "peak": fma_peak, "unit": "TFLOP/s",
        "frac": cflop / (t_c * 1e-3) / 1e12 / fma_peak,
        "peak_source": "measured in this run: tm_fma_peak (dependent-chain FFMA / FFMA2 microbenchmark, 2 flop per FMA lane)",
        "algorithmic_flop_per_site": CONTRACT_FLOP_PER_SITE, "algorithmic_bytes_per_site": CONTRACT_BYTES_PER_SITE,
        "hbm_GBps": cbytes / (t_c * 1e-3) / 1e9, "hbm_frac": cbytes / (t_c * 1e-3) / 1e9 / peak,
        "traffic": ctraffic, "traffic_source": ctraffic_src,
        "fp64_ms_per_source": t_c64,
        "paper": "~300 GFlops double precision on one Tesla M2070 (PAPER.md:84): context, another machine"}

    it_lp = np.mean([i["iters_lp"] for i in infos])
    it_hp = np.mean([i["iters_hp"] for i in infos])
    free_b, total_b = torch.cuda.mem_get_info()
    extras = {
        "hbm_in_use_gb": (total_b - free_b) / 1e9,     # gauge copies + 2 lanes x 8 sources of solver workspaces + noise
        "dslash": ds,
        "lp_iters_per_source": it_lp / max(1, n_lp), "hp_iters_per_source": it_hp / max(1, n_hp),
        "lp_cg_iters_per_sec": it_lp / (np.mean([i["ms_lp_solve"] for i in infos]) * 1e-3),
        "hp_cg_iters_per_sec": it_hp / max(1e-9, np.mean([i["ms_hp_solve"] for i in infos]) * 1e-3),
        "ms_lp_solve": float(np.mean([i["ms_lp_solve"] for i in infos])),
        "ms_hp_solve": float(np.mean([i["ms_hp_solve"] for i in infos])),
        "ms_contract_and_rest": float(np.mean([i["ms_contract"] for i in infos])),
        "lanes": int(infos[0]["lanes"]),
        "one_lane_breakdown": breakdown,
        "worst_resid_lp": max(i["worst_resid_lp"] for i in infos),
        "worst_resid_hp": max(i["worst_resid_hp"] for i in infos),
        "fp32_fma_peak_tflops": {"ffma": ctx.tm_fma_peak(0, 8192), "ffma2": ctx.tm_fma_peak(1, 8192)},
    }
    ctx.close()
    del ctx, U
    torch.cuda.empty_cache()
    if world == 1 and not args.no_c5_sweep:
        extras["c5_sweep"] = c5_sweep(tmod, torch, inputs_torch, local, peak)
        torch.cuda.empty_cache()
    line = {"metric": "tsm_sources_per_sec", "value": value, "unit": "sources/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": args.scaling, "vs_baseline": None, "dtype": "f16 storage / f32 accumulate (LP), f32+f64 (HP)",
            "data": "synthetic", "config": workload_config(cfg, args), "clocks": clocks, "e2e": e2e,
            "gpu_launches": int(launches), "roofline": roofline, "roofline_contract": roofline_contract, "extras": extras}
    if world == 1 and not args.no_cpu_baseline:
        smp = oracle_sample(cfg, hp=True)
        line["cpu_baseline"] = {
            "value": oracle_rate(cfg, smp, smp["hp_s"]), "unit": "sources/s", "cores": cores_used(), "kind": "oracle",
            "sample": "1 of %d LP solves (fp64 CGNR to rho=1e-2: %d iterations, %.1f s) + 1 of %d HP solves (rho=1e-8: %d "
                      "iterations, %.1f s) + contraction/projection of 1 of %d timeslices (%.2f s), extrapolated to the "
                      "whole step (%d + %d solves, %d contractions)"
                      % (cfg["n_lp"], smp["lp_iters"], smp["lp_s"], cfg["n_hp"], smp["hp_iters"], smp["hp_s"], dims[3],
                         smp["contract_s_per_timeslice"], cfg["n_lp"], cfg["n_hp"], cfg["n_lp"] + cfg["n_hp"]),
            "without_hp_corrections": oracle_rate(cfg, smp, None)}
        line["cpu_baseline"].update(oracle_extras(cfg))
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", default="c4", choices=["c1", "c3", "c4"])
    ap.add_argument("--scaling", default="strong", choices=["strong", "weak"],
                    help="N > 1: shard the one (N_LP, N_HP) workload over the ranks (strong) or run N times the workload (weak)")
    ap.add_argument("--what", default="step", choices=["step", "dslash", "dslash_group", "contract", "blas", "solve"],
                    help="step: the bench line; otherwise run one kernel family a few times (ncu captures)")
    ap.add_argument("--contract-path", type=int, default=0, choices=[0, 1, 2, 3, 4],
                    help="TM_OPT_CONTRACT_PATH of the fp32 contraction (0 = automatic, see include/tmloops.h)")
    ap.add_argument("--prec", default="f16", help="--what != step: storage precision (contract: f32 | f64)")
    ap.add_argument("--recon", type=int, default=12)
    ap.add_argument("--napp", type=int, default=6)
    ap.add_argument("--n-lp", type=int, default=None, help="override N_LP (debugging; invalidates the headline)")
    ap.add_argument("--n-hp", type=int, default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--step-only", action="store_true",
                    help="warm-up + timed TSM steps only (no end-to-end leg, rooflines, sweep or CPU baseline): the command of "
                         "the ncu launch list under profiles/")
    ap.add_argument("--no-c5-sweep", action="store_true")
    ap.add_argument("--lp-delta", type=float, default=None, help="reliable-update trigger of the LP solves (tuning)")
    ap.add_argument("--hp-delta", type=float, default=None, help="reliable-update trigger of the HP solves (tuning)")
    args = ap.parse_args()
    cfg = dict(inputs.CONFIGS[args.config])
    cfg.setdefault("n_lp", 4)
    cfg.setdefault("n_hp", 2)
    cfg.setdefault("p2max", 0)
    if args.n_lp is not None:
        cfg["n_lp"] = args.n_lp
    if args.n_hp is not None:
        cfg["n_hp"] = args.n_hp
    if args.lp_delta is not None:
        LP["delta"] = args.lp_delta
    if args.hp_delta is not None:
        HP["delta"] = args.hp_delta
    if args.impl == "reference":
        run_reference(args, cfg)
    elif args.what != "step":
        profile_mode(args, cfg)
    else:
        run_b200(args, cfg)


if __name__ == "__main__":
    main()
