"""Run one hot kernel family a few times on paper-sized fields (for ncu captures).

    python -m paper_1401_6750_b200.profile_kernels --what dslash --prec f16 --recon 12 --dims 32 32 32 64 --napp 6
    python -m paper_1401_6750_b200.profile_kernels --what contract --prec f32 --dims 32 32 32 64
    python -m paper_1401_6750_b200.profile_kernels --what solve --prec f16 --dims 32 32 32 64

Prints CUDA-event timings; meant to be wrapped as `<cmd> && ncu ... <cmd>` (B200_PROFILING.md).
"""
from __future__ import annotations

import argparse

import torch

import paper_1401_6750_b200 as tmod
from paper_1401_6750_b200 import inputs, inputs_torch


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--what", default="dslash", choices=["dslash", "contract", "solve", "sweep"])
    ap.add_argument("--prec", default="f16")
    ap.add_argument("--recon", type=int, default=12)
    ap.add_argument("--dims", type=int, nargs=4, default=[32, 32, 32, 64])
    ap.add_argument("--napp", type=int, default=6)
    ap.add_argument("--op", default="XPAY")
    ap.add_argument("--nb", type=int, default=1, help="dslash: sources per launch (tm_dslash_multi)")
    ap.add_argument("--eps", type=float, default=0.2)
    ap.add_argument("--kappa", type=float, default=0.161231)
    ap.add_argument("--mu", type=float, default=0.004)
    ap.add_argument("--p2max", type=int, default=9)
    a = ap.parse_args()
    dims = tuple(a.dims)
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    U = inputs_torch.gauge_field(dims, a.eps, 5, dev)
    ctx = tmod.TmContext(dims, -1, 0)
    ctx.tm_load_gauge(U)
    del U
    P = tmod.PREC[a.prec]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if a.what == "dslash":
        tdt = {"f64": torch.float64, "f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}[a.prec]
        nb = 3
        pb = ctx.tm_field_bytes(P, False)
        ins = [torch.empty(a.nb * pb, dtype=torch.uint8, device=dev) for _ in range(nb)]
        outs = [torch.empty(a.nb * pb, dtype=torch.uint8, device=dev) for _ in range(nb)]
        xs = torch.empty(a.nb * pb, dtype=torch.uint8, device=dev)
        for b in ins + [xs]:
            v = b.view(tdt)
            v.copy_((torch.rand(v.shape, device=dev, dtype=torch.float32) - 0.5).to(tdt))
        op = getattr(tmod, "TM_OP_" + a.op)

        def launch(i):
            if a.nb == 1:
                ctx.tm_dslash(outs[i % nb], ins[i % nb], xs, op, 0, False, a.kappa, a.mu, P, a.recon)
            else:
                ctx.tm_dslash_multi(outs[i % nb], ins[i % nb], xs, a.nb, op, 0, False, a.kappa, a.mu, P)
        for i in range(3):
            launch(i)
        torch.cuda.synchronize()
        e0.record()
        for i in range(a.napp):
            launch(i)
        e1.record()
        torch.cuda.synchronize()
        V = inputs.volume(dims)
        us = e0.elapsed_time(e1) * 1e3 / a.napp
        xb = 24 if a.op == "XPAY" else 0
        nbytes = (a.nb * (48 + xb) + 8 * a.recon) * tmod.PREC_BYTES[P] * (V // 2)
        print("dslash %s r%d %s, %d source(s) per launch: %.1f us/launch, %.0f GB/s (spinors per source, links once per launch)"
              % (a.prec, a.recon, a.op, a.nb, us, nbytes / us / 1e3))
    elif a.what == "sweep":
        # BASELINE.json configs[4] (bandwidth sweep): standalone parity Dslash (XPAY epilogue) and one CG iteration
        # (4 Dslash + fused BLAS-1) per storage precision / reconstruct; a.napp applications each
        import json
        import os
        V = inputs.volume(dims)
        Vh = V // 2
        pk = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "MEASURED_PEAKS.json")
        peak = json.load(open(pk))["hbm_gbs"] if os.path.exists(pk) else 6650.0
        print("| storage | recon | us / Dslash | GB/s (algorithmic) | frac of %.0f GB/s | GFLOP/s | CG it/s | us / CG iteration |" % peak)
        print("|---|---|---|---|---|---|---|---|")
        eta = inputs_torch.z4_source(dims, 11, 0, dev)
        for prec in ("f64", "f32", "f16", "bf16"):
            for recon in (12, 18):
                Pq = tmod.PREC[prec]
                tdt = {"f64": torch.float64, "f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}[prec]
                nb = 3
                ins = [ctx.empty_field(Pq, False) for _ in range(nb)]
                outs = [ctx.empty_field(Pq, False) for _ in range(nb)]
                xs = ctx.empty_field(Pq, False)
                for b in ins + [xs]:
                    v = b.view(tdt)
                    v.copy_((torch.rand(v.shape, device=dev, dtype=torch.float32) - 0.5).to(tdt))
                for i in range(5):
                    ctx.tm_dslash(outs[i % nb], ins[i % nb], xs, tmod.TM_OP_XPAY, 0, False, a.kappa, a.mu, Pq, recon)
                torch.cuda.synchronize()
                e0.record()
                for i in range(a.napp):
                    ctx.tm_dslash(outs[i % nb], ins[i % nb], xs, tmod.TM_OP_XPAY, 0, False, a.kappa, a.mu, Pq, recon)
                e1.record()
                torch.cuda.synchronize()
                us = e0.elapsed_time(e1) * 1e3 / a.napp
                gbs = (48 + 8 * recon + 24) * tmod.PREC_BYTES[Pq] * Vh / us / 1e3
                del ins, outs, xs
                # CG: a fixed number of iterations (rho unreachable, max_iter = 40) so that it/s is per iteration
                outer = "f32" if prec in ("f16", "bf16") else prec
                for i in range(2):
                    s, info = ctx.tm_cg_solve(eta, a.kappa, a.mu, prec, outer, recon, 1e-30, 40, 1e-30, raise_on_noconv=False)
                it_us = info["ms"] * 1e3 / max(1, info["iters"])
                print("| %s | %d | %.1f | %.0f | %.2f | %.0f | %.0f | %.1f |" % (
                    prec, recon, us, gbs, gbs / peak, 1416.0 * Vh / us / 1e3, 1e6 / it_us, it_us))
    elif a.what == "contract":
        s = inputs_torch.z4_source(dims, 11, 0, dev)
        eta = inputs_torch.z4_source(dims, 11, 1, dev)
        mom = inputs.momentum_list(a.p2max)
        ctx.loop_contract_project(s, eta, a.kappa, a.mu, mom, P)
        torch.cuda.synchronize()
        e0.record()
        for i in range(a.napp):
            ctx.loop_contract_project(s, eta, a.kappa, a.mu, mom, P)
        e1.record()
        torch.cuda.synchronize()
        print("contract %s: %.3f ms/call (includes 2 canonical->internal imports)" % (a.prec, e0.elapsed_time(e1) / a.napp))
    else:
        eta = inputs_torch.z4_source(dims, 11, 0, dev)
        outer = "f32" if a.prec in ("f16", "bf16") else "f64"
        rho = 1e-2 if outer == "f32" else 1e-8
        for i in range(2):
            s, info = ctx.tm_cg_solve(eta, a.kappa, a.mu, a.prec, outer, a.recon, rho, 5000)
        print("solve %s/%s rho=%g: %s" % (a.prec, outer, rho, info))
    ctx.close()


if __name__ == "__main__":
    main()
