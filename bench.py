#!/usr/bin/env python
"""bench.py -- TSM sources/sec at 32^3x64 (BASELINE.json metric) on B200, with the Dslash roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference] [--config c4]

One "step" = one pass of the whole hot path over one batch of synthetic input: the full TSM
estimator loop of BASELINE.json config c4 (N_LP = 500 Z4 sources solved with 16-bit storage to
rho = 1e-2, N_HP = 20 of them solved mixed fp32/fp64 to rho = 1e-8, every solution contracted into
the 160 insertions and projected onto the 123 momenta with p^2 <= 9 for all 64 timeslices).
`value` = N_LP sources / step time, inputs (gauge field, packed Z4 noise) resident in HBM.
`e2e` = the same through the host-buffer entry point: gauge field and packed noise start in pinned
host memory, the estimate ends in pinned host memory, all copies inside the timed region.
N > 1 (torchrun): sources are sharded by rank (weak scaling: every rank runs the c4 workload on
its own noise streams), the only exchange is one all-reduce of the 20 MB estimate per step.

`--impl reference` times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the
same workload on the host cores; see cpu_baseline in the JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1401_6750_b200 import inputs  # noqa: E402

LP = dict(sloppy="f16", outer="f32", recon=12, rho=1e-2, max_iter=2000, delta=0.01)
HP = dict(sloppy="f32", outer="f64", recon=12, rho=1e-8, max_iter=5000, delta=0.01)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic(prec, suffix=""):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed
    `ncu --set full` summary (text) of the same kernel, or None when no capture of it is committed."""
    import re
    p = os.path.join(ROOT, "profiles", "r01_dslash16_%s%s.md" % (prec, suffix))
    if not os.path.exists(p):
        return None, None
    tot, scale = 0.0, {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    for m in re.finditer(r"`dram__bytes_(?:read|write)\.sum` \| ([0-9.,]+) \| (\w+)", open(p).read()):
        tot += float(m.group(1).replace(",", "")) * scale[m.group(2)]
    return (tot or None), "profiles/" + os.path.basename(p)


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
def oracle_sample(cfg, n_timeslices=1):
    """Bounded sample of the c4 workload on the host cores with the oracle AS IT STANDS:
    one LP solve (rho = 1e-2, fp64 CGNR) + contraction/projection of n_timeslices of T timeslices
    (extrapolated x T/n).  HP corrections are not included (they would only make it slower)."""
    import oracle  # test infrastructure; allowed in bench.py's cpu_baseline / --impl reference legs only
    oracle.build()
    dims = cfg["dims"]
    U = oracle_inputs_cache(cfg)
    eta = inputs.z4_source(dims, cfg["src_seed"], 0)
    mom = inputs.momentum_list(cfg.get("p2max", 9))
    t0 = time.perf_counter()
    s, iters, tr, st = oracle.solve(eta, U, cfg["kappa"], cfg["mu"], LP["rho"])
    t1 = time.perf_counter()
    oracle.loops_project(s, eta, U, cfg["kappa"], cfg["mu"], mom, -1, 0, n_timeslices)
    t2 = time.perf_counter()
    T = dims[3]
    sec_per_source = (t1 - t0) + (t2 - t1) * T / n_timeslices
    return dict(sec_per_source=sec_per_source, solve_s=t1 - t0, iters=iters, true_resid=tr,
                contract_s_per_timeslice=(t2 - t1) / n_timeslices)


_U_CACHE = {}


def oracle_inputs_cache(cfg):
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


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    times, last = [], None
    for i in range(args.warmup + args.steps):
        last = oracle_sample(cfg)
        if i >= args.warmup:
            times.append(last["sec_per_source"])
    sec = float(np.mean(times)) if times else last["sec_per_source"]
    val = 1.0 / sec
    sample = ("per step: 1 of %d LP sources (oracle fp64 CGNR to rho=1e-2, %d iterations) + contraction/projection of "
              "1 of %d timeslices, extrapolated; HP corrections excluded" % (cfg["n_lp"], last["iters"], cfg["dims"][3]))
    line = {"impl": "reference", "metric": "tsm_sources_per_sec", "value": val, "unit": "sources/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * cfg["n_lp"] * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
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
            "sources_counted": "n_lp per step per GPU",
            "l2": "working set (gauge 201 MB 16-bit / 403 MB fp32 + vectors) exceeds the 126 MB L2; Dslash microbench "
                  "rotates over 4 field pairs",
            "parallelism": "sources sharded by rank, one all-reduce of the estimate per step"}


# ----------------------------------------------------------------------------- CUDA arm
def time_dslash(ctx, tmod, torch, prec, recon, kappa, mu, napp, op_name="XPAY"):
    """Average CUDA-event time of one parity-Dslash launch (16-byte vector internal layout)."""
    P = tmod.PREC[prec]
    nb = 4
    ins = [ctx.empty_field(P, False) for _ in range(nb)]
    outs = [ctx.empty_field(P, False) for _ in range(nb)]
    xs = ctx.empty_field(P, False)
    # fill with a valid field: Gaussian numbers via import of a random canonical spinor would cost
    # 400 MB of host->device traffic; a device-side uniform fill in storage precision is enough
    # (Dslash cost is data-independent)
    tdt = {"f64": torch.float64, "f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}[prec]
    g = torch.Generator(device=ctx.tdev)
    g.manual_seed(1234)
    for b in ins + [xs]:
        v = b.view(tdt)
        v.copy_((torch.rand(v.shape, generator=g, device=ctx.tdev, dtype=torch.float32) - 0.5).to(tdt))
    op = getattr(tmod, "TM_OP_" + op_name)
    for i in range(8):
        ctx.tm_dslash(outs[i % nb], ins[i % nb], xs, op, 0, False, kappa, mu, P, recon)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(napp):
        ctx.tm_dslash(outs[i % nb], ins[i % nb], xs, op, 0, False, kappa, mu, P, recon)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / napp


def time_dslash_multi(ctx, tmod, torch, prec, nb, kappa, mu, napp):
    """Average CUDA-event time of one nb-source parity-Dslash launch (XPAY, reconstruct-12), as tsm_estimate launches it."""
    P = tmod.PREC[prec]
    pb = ctx.tm_field_bytes(P, False)
    tdt = {"f64": torch.float64, "f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}[prec]
    nbuf = 3
    ins = [torch.empty(nb * pb, dtype=torch.uint8, device=ctx.tdev) for _ in range(nbuf)]
    outs = [torch.empty(nb * pb, dtype=torch.uint8, device=ctx.tdev) for _ in range(nbuf)]
    xs = torch.empty(nb * pb, dtype=torch.uint8, device=ctx.tdev)
    g = torch.Generator(device=ctx.tdev)
    g.manual_seed(4321)
    for b in ins + [xs]:
        v = b.view(tdt)
        v.copy_((torch.rand(v.shape, generator=g, device=ctx.tdev, dtype=torch.float32) - 0.5).to(tdt))
    for i in range(4):
        ctx.tm_dslash_multi(outs[i % nbuf], ins[i % nbuf], xs, nb, tmod.TM_OP_XPAY, 0, False, kappa, mu, P)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(napp):
        ctx.tm_dslash_multi(outs[i % nbuf], ins[i % nbuf], xs, nb, tmod.TM_OP_XPAY, 0, False, kappa, mu, P)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / napp


def dslash_bytes_per_site(prec, recon, xpay):
    b = {"f64": 8, "f32": 4, "f16": 2, "bf16": 2}[prec]
    return (48 + 8 * recon + (24 if xpay else 0)) * b     # read 1 spinor, 8 links, write 1 (+ x)


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
    n_lp, n_hp = cfg["n_lp"], cfg["n_hp"]
    kappa, mu = cfg["kappa"], cfg["mu"]
    mom = inputs.momentum_list(cfg["p2max"])
    seed = multi.rank_seed(cfg["src_seed"], rank)

    U = inputs_torch.gauge_field(dims, cfg["eps"], cfg["seed"], dev)
    z4_dev = torch.empty((n_lp, 3 * V), dtype=torch.uint8, device=dev)
    for r in range(n_lp):
        z4_dev[r] = inputs_torch.z4_packed(dims, seed, r, dev)
    ctx = tmod.TmContext(dims, -1, local)
    ctx.tm_load_gauge(U)

    def step():
        out, _, info = ctx.tsm_estimate(n_lp, n_hp, kappa, mu, mom, LP, HP, tmod.TM_F32, tmod.TM_F64, z4=z4_dev)
        out = multi.combine_over_ranks(out, n_lp, n_hp)
        return out, info

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
    value = world * n_lp / (ms_per_step * 1e-3)

    # ---- end to end through host buffers (pinned): gauge + noise H2D, estimate D2H, every step
    U_host = torch.empty(U.shape, dtype=U.dtype).pin_memory()
    U_host.copy_(U)
    z4_host = torch.empty(z4_dev.shape, dtype=torch.uint8).pin_memory()
    z4_host.copy_(z4_dev)
    del z4_dev
    out_host = torch.empty((2, 80, len(mom), dims[3]), dtype=torch.complex128).pin_memory()
    U_stage = torch.empty_like(U)

    def e2e_step():
        U_stage.copy_(U_host, non_blocking=True)
        ctx.tm_load_gauge(U_stage)
        o, info = ctx.tsm_estimate_host(n_lp, n_hp, kappa, mu, mom, LP, HP, tmod.TM_F32, tmod.TM_F64,
                                        z4_host=z4_host, out_host=out_host)
        if world > 1:
            g = multi.combine_over_ranks(o.to(dev), n_lp, n_hp)
            o.copy_(g)
        return o

    e2e_step()
    barrier()
    e2e_steps = max(1, min(args.steps, 2))
    w0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    barrier()
    e2e_s = torch.tensor([(time.perf_counter() - w0) / e2e_steps], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(e2e_s, op=dist.ReduceOp.MAX)
    e2e = {"value": world * n_lp / float(e2e_s.item()), "unit": "sources/s",
           "h2d_bytes_per_step": int(U_host.numel() * 16 + z4_host.numel()),
           "d2h_bytes_per_step": int(out_host.numel() * 16), "steps": e2e_steps,
           "timing": "host wall clock around the synchronous host-buffer call, max over ranks"}
    del U_host, z4_host, U_stage

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- dominant kernel: the 16-bit parity Dslash with fused XPAY epilogue (timed alone -> burst peak)
    peak, peak_src = peaks()
    Vh = V // 2
    napp = 200
    ds = {}
    for prec, recon in (("f16", 12), ("bf16", 12), ("f16", 18), ("f32", 12), ("f64", 12)):
        t_ms = time_dslash(ctx, tmod, torch, prec, recon, kappa, mu, napp)
        nbytes = dslash_bytes_per_site(prec, recon, True) * Vh
        ds[prec + "_r%d" % recon] = {"us": t_ms * 1e3, "GBps": nbytes / (t_ms * 1e-3) / 1e9,
                                     "GFLOPs": (1320 + 96) * Vh / (t_ms * 1e-3) / 1e9}
    dom = ds[LP["sloppy"] + "_r12"]
    roofline = {"bound": "hbm", "kernel": "dslash16_kernel<%s> reconstruct-12 XPAY (second half of Mhat), one source per launch" % LP["sloppy"],
                "achieved": dom["GBps"], "peak": peak, "unit": "GB/s", "frac": dom["GBps"] / peak,
                "traffic": None, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": dslash_bytes_per_site(LP["sloppy"], 12, True) * Vh,
                "how": "CUDA events around %d back-to-back launches on the current stream, 4 rotating field pairs" % napp}
    roofline["traffic"], roofline["traffic_source"] = ncu_traffic(LP["sloppy"])
    # the same kernel as tsm_estimate launches it: GROUP sources per launch, links read from HBM once per group
    # (later readers hit L2).  Two accountings: the bytes such a launch must move (spinors per source, links once),
    # and the single-source equivalent (SURVEY.md sec 8d bytes per site x sites x sources).
    GROUP = 8
    t_g = time_dslash_multi(ctx, tmod, torch, LP["sloppy"], GROUP, kappa, mu, 60)
    b16 = 2
    must_move = (GROUP * (48 + 24) + 8 * 12) * b16 * Vh
    roofline["grouped"] = {
        "sources_per_launch": GROUP, "us_per_launch": t_g * 1e3, "us_per_source": t_g * 1e3 / GROUP,
        "hbm_bytes_per_launch": must_move, "achieved_GBps": must_move / (t_g * 1e-3) / 1e9,
        "frac_of_peak": must_move / (t_g * 1e-3) / 1e9 / peak,
        "single_source_equivalent_GBps": GROUP * dslash_bytes_per_site(LP["sloppy"], 12, True) * Vh / (t_g * 1e-3) / 1e9,
        "traffic": ncu_traffic(LP["sloppy"], "_group8")[0],
        "note": "not HBM-bound any more: limited by instruction issue and board power (DESIGN.md sec 6)"}

    it_lp = np.mean([i["iters_lp"] for i in infos])
    it_hp = np.mean([i["iters_hp"] for i in infos])
    free_b, total_b = torch.cuda.mem_get_info()
    extras = {
        "hbm_in_use_gb": (total_b - free_b) / 1e9,     # gauge copies + 2 lanes x 8 sources of solver workspaces + noise
        "dslash": ds,
        "lp_iters_per_source": it_lp / n_lp, "hp_iters_per_source": it_hp / max(1, n_hp),
        "lp_cg_iters_per_sec": it_lp / (np.mean([i["ms_lp_solve"] for i in infos]) * 1e-3),
        "hp_cg_iters_per_sec": it_hp / max(1e-9, np.mean([i["ms_hp_solve"] for i in infos]) * 1e-3),
        "ms_lp_solve": float(np.mean([i["ms_lp_solve"] for i in infos])),
        "ms_hp_solve": float(np.mean([i["ms_hp_solve"] for i in infos])),
        "ms_contract_and_rest": float(np.mean([i["ms_contract"] for i in infos])),
        "worst_resid_lp": max(i["worst_resid_lp"] for i in infos),
        "worst_resid_hp": max(i["worst_resid_hp"] for i in infos),
    }
    line = {"metric": "tsm_sources_per_sec", "value": value, "unit": "sources/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f16 storage / f32 accumulate (LP), f32+f64 (HP)",
            "data": "synthetic", "config": workload_config(cfg, args), "clocks": clocks, "e2e": e2e,
            "gpu_launches": int(launches), "roofline": roofline, "extras": extras}
    if world == 1 and not args.no_cpu_baseline:
        del U
        torch.cuda.empty_cache()
        smp = oracle_sample(cfg)
        line["cpu_baseline"] = {
            "value": 1.0 / smp["sec_per_source"], "unit": "sources/s", "cores": cores_used(), "kind": "oracle",
            "sample": "1 of %d LP sources (fp64 CGNR to rho=1e-2: %d iterations, %.1f s) + contraction/projection of 1 of %d "
                      "timeslices (%.1f s), extrapolated; HP corrections excluded"
                      % (n_lp, smp["iters"], smp["solve_s"], dims[3], smp["contract_s_per_timeslice"])}
    print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", default="c4", choices=["c1", "c3", "c4"])
    ap.add_argument("--n-lp", type=int, default=None, help="override N_LP (debugging; invalidates the headline)")
    ap.add_argument("--n-hp", type=int, default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
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
    else:
        run_b200(args, cfg)


if __name__ == "__main__":
    main()
