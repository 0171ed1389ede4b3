// solver.cu -- eq. 2.1: M s = eta by even-odd preconditioned CG on Mhat^dag Mhat
// (SURVEY.md sec 8 rows a2-a5).  CGLS recurrences in `sloppy` storage, x and r accumulated in
// >= fp32, reliable updates and the final true-residual test in `outer` precision.
//
//   Mhat   = A - kappa^2 D_eo A^-1 D_oe            (A = 1 + 2 i kappa mu g5)
//   bhat_e = eta_e + kappa D_eo A^-1 eta_o
//   s_o    = A^-1 (eta_o + kappa D_oe s_e)
// With s_o reconstructed this way eta - M s vanishes on odd sites and equals bhat - Mhat s_e on even
// sites, so ||bhat - Mhat y|| / ||eta|| evaluated in `outer` precision IS the true residual.
//
// Control flow lives on the device (blas.cuh, CgScalars): the last block of every reducing kernel
// computes alpha / beta, decides when to pause for a reliable update and when the solve is over;
// every kernel is guarded by that state.  The host only enqueues:
//   iteration block  (GUARD_ITER)  z = Mhat^dag r ; p = z + beta p ; w = Mhat p ; x += alpha p, r -= alpha w
//   update block     (GUARD_RU)    y += x, x = 0 ; r = bhat - Mhat y in outer precision ; resume | finish
//   tail             (always)      s_o = A^-1 eta_o + kappa [A^-1 D_oe y]   (bracket: by-product of the last update)
// along the plan recorded by the previous solve with the same parameters, and reads the state back
// once at the end (one host synchronisation per solve when the plan fits; otherwise it keeps
// enqueueing [iteration, update] pairs and polls).
#include <math.h>
#include "kernels.h"

// out = Mhat in (dagger: Mhat^dag in) on even sites; tmp: odd-parity scratch of the same precision
// in_mul: source stride of `in` in parity vectors (2 when `in` is the even half of a full-lattice field)
static tm_status apply_mhat(tm_ctx* ctx, void* out, const void* in, void* tmp, int dagger, double kappa,
                            double mu, tm_prec prec, tm_recon recon, int red_op, int guard, cudaStream_t st,
                            int in_mul = 1) {
    DslashCall k;
    memset(&k, 0, sizeof(k));
    k.kappa = kappa; k.mu = mu; k.dagger = dagger; k.guard = guard;
    k.out = tmp; k.in = in; k.out_parity = 1; k.post = 1; k.coef = 1.0; k.red_op = RED_NONE;
    k.mul_in = in_mul;
    TM_TRY(tm_dslash_launch(ctx, k, prec, recon, st));
    k.out = out; k.in = tmp; k.x = in; k.out_parity = 0; k.post = 0; k.xmode = 2; k.coef = -kappa * kappa;
    k.mul_in = 1; k.mul_x = in_mul;
    k.red_op = red_op;
    return tm_dslash_launch(ctx, k, prec, recon, st);
}

// One solve in two host phases, so that several solves can be in flight on different lanes (tsm.cu):
//   tm_solve_begin  enqueues setup + the planned iteration / update blocks + tail + an asynchronous
//                   download of the device state, without any host synchronisation;
//   tm_solve_end    waits for that download, continues off plan if the state machine has not finished,
//                   records the plan of the next solve and fills `info`.
// Both must be called with the same lane of the context active (tm_lane_use).
static tm_status job_iteration(tm_ctx* ctx, const SolveJob& J) {
    TM_TRY(apply_mhat(ctx, J.z, J.rs, J.tmp, 1, J.kappa, J.mu, J.ps, J.rc, RED_ZZ, GUARD_ITER, J.st));
    TM_TRY(blas_update_p(ctx, J.p, J.z, J.ps, J.x, J.pa, J.st));
    TM_TRY(apply_mhat(ctx, J.w, J.p, J.tmp, 0, J.kappa, J.mu, J.ps, J.rc, RED_WW, GUARD_ITER, J.st));
    return blas_update_xr(ctx, J.r, J.pa, J.w, J.rs, J.ps, J.st);
}
static tm_status job_update(tm_ctx* ctx, const SolveJob& J) {
    TM_TRY(blas_ru_begin(ctx, J.y, J.po, J.x, J.pa, J.p, J.ps, J.st, 2));
    TM_TRY(apply_mhat(ctx, J.mo, J.y, J.tmpo, 0, J.kappa, J.mu, J.po, J.rc, RED_NONE, GUARD_RU, J.st, 2));
    return blas_residual(ctx, J.r, J.pa, J.rs, J.ps, J.b, J.mo, J.po, RED_RU, GUARD_RU, J.st);
}
// s_o = A^-1 (eta_o + kappa D_oe y) = A^-1 eta_o + kappa [A^-1 D_oe y]: the bracket is the first half of Mhat y,
// left in tmpo by the LAST reliable update that ran -- and the solve always ends on one (it is the update that
// declares convergence or failure; y does not change after it), so the tail needs no Dslash of its own.
static tm_status job_tail(tm_ctx* ctx, const SolveJob& J) {
    TM_TRY(blas_twist_inv_axpy(ctx, J.s_o, J.eta_o, J.tmpo, J.po, J.kappa, J.mu, J.kappa, J.st, 2, 2, 1));
    TM_CUDA(ctx, cudaEventRecord(J.e1, J.st));
    return TM_OK;
}

// Launch plans are keyed by the whole parameter tuple, so LP and HP solves that share a sloppy precision (or two
// parameter sets used alternately) keep their own plan instead of evicting each other's on every pass.
static bool plan_matches(const CgPlan& p, const SolveJob& J) {
    return p.valid && p.sloppy == (int)J.ps && p.outer == (int)J.po && p.recon == (int)J.rc
        && p.max_iter == J.P.max_iter && p.rho == J.P.rho && p.delta == J.delta;
}
static CgPlan* find_plan(tm_ctx* ctx, const SolveJob& J) {
    for (int i = 0; i < TM_NPLANS; i++)
        if (plan_matches(ctx->plan[i], J)) return &ctx->plan[i];
    return nullptr;
}
static CgPlan* plan_slot(tm_ctx* ctx, const SolveJob& J) {
    CgPlan* p = find_plan(ctx, J);
    if (p) return p;
    for (int i = 0; i < TM_NPLANS; i++)
        if (!ctx->plan[i].valid) return &ctx->plan[i];
    p = &ctx->plan[ctx->plan_next];
    ctx->plan_next = (ctx->plan_next + 1) % TM_NPLANS;
    return p;
}

// every launcher reads ctx->nb; it is 2 only while a paired solve enqueues
struct NbScope {
    tm_ctx* c;
    NbScope(tm_ctx* ctx, int nb) : c(ctx) { c->nb = nb; }
    ~NbScope() { c->nb = 1; }
};

tm_status tm_solve_begin(tm_ctx* ctx, SolveJob* Jp, void* d_s, const void* d_eta, double kappa, double mu,
                         const tm_solve_params* P, cudaStream_t st, double eta_norm2, int nb) {
    SolveJob& J = *Jp;
    if (!P) return tm_fail(ctx, TM_EARG, "solve: null params");
    if (nb < 1 || nb > TM_MAXNB || (nb & (nb - 1))) return tm_fail(ctx, TM_EARG, "solve: nb must be a power of two <= TM_MAXNB");
    if (nb > 1 && !(eta_norm2 > 0)) return tm_fail(ctx, TM_EARG, "solve: a grouped solve needs the source norm");
    J.nb = nb;
    NbScope scope(ctx, nb);
    const tm_prec po = P->outer, ps = P->sloppy;
    if (po != TM_F64 && po != TM_F32) return tm_fail(ctx, TM_EPREC, "solve: outer precision must be f32 or f64");
    if ((int)ps < 0 || (int)ps > 3) return tm_fail(ctx, TM_EPREC, "solve: unknown sloppy precision");
    if (tm_prec_size(ps) > tm_prec_size(po)) return tm_fail(ctx, TM_EPREC, "solve: sloppy precision wider than outer");
    if (P->recon != TM_R12 && P->recon != TM_R18) return tm_fail(ctx, TM_EARG, "solve: recon must be 12 or 18");
    if (!(P->rho > 0) || P->max_iter < 0) return tm_fail(ctx, TM_EARG, "solve: rho must be > 0, max_iter >= 0");
    J.P = *P;
    J.po = po; J.ps = ps;
    J.pa = (ps == TM_F64) ? TM_F64 : TM_F32;        // accumulate precision of x, r
    J.rc = P->recon;
    J.delta = (P->delta > 0 && P->delta < 1) ? P->delta : 0.1;
    J.kappa = kappa; J.mu = mu; J.st = st;
    // workspaces of a pair keep source 1's vector right behind source 0's (stride 1 parity vector); the full-lattice
    // fields d_eta / d_s keep each source's [even][odd] contiguous (stride 2 parity vectors: the *_mul = 2 operands)
    const size_t bo1 = tm_parity_bytes(ctx, po);
    const size_t bo = nb * bo1, bs = nb * tm_parity_bytes(ctx, ps), ba = nb * tm_parity_bytes(ctx, J.pa);

    J.e0 = ctx->ev[0]; J.e1 = ctx->ev[1];
    TM_CUDA(ctx, cudaEventRecord(J.e0, st));

    TM_TRY(tm_ws(ctx, WS_SL_P, bs, &J.p));
    TM_TRY(tm_ws(ctx, WS_SL_W, bs, &J.w));
    TM_TRY(tm_ws(ctx, WS_SL_Z, bs, &J.z));
    TM_TRY(tm_ws(ctx, WS_SL_TMP, bs, &J.tmp));
    TM_TRY(tm_ws(ctx, WS_AC_X, ba, &J.x));
    // fp16 sloppy storage: the iterated residual lives in fp16 only (11-bit mantissa: 2.4e-4 relative rounding per
    // update, far below what a reliable update corrects); bf16 (8 bits) keeps an fp32 copy
    if (ps == TM_F16) J.r = nullptr; else TM_TRY(tm_ws(ctx, WS_AC_R, ba, &J.r));
    if (J.pa != ps) TM_TRY(tm_ws(ctx, WS_SL_R, bs, &J.rs)); else J.rs = J.r;
    TM_TRY(tm_ws(ctx, WS_OU_B, bo, &J.b));
    TM_TRY(tm_ws(ctx, WS_OU_TMP, bo, &J.tmpo));
    TM_TRY(tm_ws(ctx, WS_OU_TMP2, bo, &J.mo));

    const char* eta_e = (const char*)d_eta;
    J.eta_o = eta_e + bo1;
    J.y = (char*)d_s;                      // the even half of the solution is accumulated in place
    J.s_o = J.y + bo1;

    // ---- setup (no host synchronisation): state (x and y zero by construction: CgScalars::x_zero / y_zero), ||eta||^2,
    //      bhat, r = rs = bhat
    TM_TRY(scal_init(ctx, P->rho * P->rho, J.delta * J.delta, P->max_iter, eta_norm2 > 0 ? eta_norm2 : 0.0, st));
    if (!(eta_norm2 > 0)) TM_TRY(blas_norm_full(ctx, d_eta, po, RED_SLOT0 + 0, st));
    TM_TRY(blas_twist_inv(ctx, J.tmpo, J.eta_o, po, kappa, mu, 0, st, 1, 2));
    {
        DslashCall k;
        memset(&k, 0, sizeof(k));
        k.out = J.b; k.in = J.tmpo; k.x = eta_e; k.out_parity = 0; k.kappa = kappa; k.mu = mu;
        k.xmode = 1; k.coef = kappa; k.red_op = RED_NONE; k.mul_x = 2;
        TM_TRY(tm_dslash_launch(ctx, k, po, J.rc, st));
    }
    TM_TRY(blas_residual(ctx, J.r, J.pa, J.rs, ps, J.b, nullptr, po, RED_START, GUARD_ALWAYS, st));

    const CgPlan* planp = find_plan(ctx, J);
    const bool have_plan = planp != nullptr;
    CgPlan plan_copy;
    if (have_plan) plan_copy = *planp;
    const CgPlan& plan = plan_copy;
    J.tail_valid = false;
    J.enq = 0;                                      // iteration blocks enqueued so far
    if (have_plan) {
        for (int k = 0; k < plan.n_pause; k++) {
            for (; J.enq < plan.pause_iter[k]; J.enq++) TM_TRY(job_iteration(ctx, J));
            TM_TRY(job_update(ctx, J));
        }
        TM_TRY(job_tail(ctx, J));
        J.tail_valid = true;
    } else {
        TM_TRY(job_update(ctx, J));                 // covers "already converged at x = 0" (state 1 after RED_START)
    }
    J.h_scal = ctx->h_scal;
    J.e_scal = ctx->ev[4];
    TM_CUDA(ctx, cudaMemcpyAsync(ctx->h_scal, ctx->d_scal, TM_MAXNB * sizeof(CgScalars), cudaMemcpyDeviceToHost, st));
    TM_CUDA(ctx, cudaEventRecord(J.e_scal, st));
    return TM_OK;
}

// info: array of J.nb entries (may be NULL).  TM_ENOCONV if any source of the job missed its rho.
tm_status tm_solve_end(tm_ctx* ctx, SolveJob* Jp, tm_solve_info* info) {
    SolveJob& J = *Jp;
    const tm_solve_params* P = &J.P;
    cudaStream_t st = J.st;
    const int nb = J.nb;
    NbScope scope(ctx, nb);
    CgScalars sc[TM_MAXNB];
    TM_CUDA(ctx, cudaEventSynchronize(J.e_scal));
    for (int b = 0; b < TM_MAXNB; b++) sc[b] = J.h_scal[b];
    auto running = [&]() {
        for (int b = 0; b < nb; b++)
            if (sc[b].done < 2) return true;
        return false;
    };
    // progress of the device state machine: every [iteration, update] pair advances a running source by one iteration
    // (state 0) or one reliable update (state 1), whatever the host had enqueued speculatively before
    auto progress = [&]() {
        long p = 0;
        for (int b = 0; b < nb; b++) p += (long)sc[b].iters + (long)sc[b].n_ru + (sc[b].done >= 2 ? 1 : 0);
        return p;
    };
    int stuck = 0;
    while (running()) {
        // off plan (first solve with these parameters, or a source behaves differently):
        // [iteration, update] pairs, polled every few pairs
        const int burst = 4;
        const long before = progress();
        for (int k = 0; k < burst; k++) { TM_TRY(job_iteration(ctx, J)); TM_TRY(job_update(ctx, J)); J.enq++; }
        J.tail_valid = false;
        TM_TRY(scal_get(ctx, sc, st));
        // failsafe on the DEVICE's own counters (not on the number of blocks enqueued, many of which the guards turn
        // into no-ops): only a state machine that did not move at all over several polls is broken
        stuck = (running() && progress() == before) ? stuck + 1 : 0;
        if (stuck >= 3) return tm_fail(ctx, TM_ECUDA, "solve: device state machine did not advance");
    }
    if (!J.tail_valid) TM_TRY(job_tail(ctx, J));
    TM_CUDA(ctx, cudaEventSynchronize(J.e1));
    // remember where this solve paused: the launch plan of the next one (a group: the union of its sources' pauses)
    CgPlan& plan = *plan_slot(ctx, J);
    plan.valid = 1;
    plan.sloppy = (int)J.ps; plan.outer = (int)J.po; plan.recon = (int)J.rc; plan.max_iter = P->max_iter;
    plan.rho = P->rho; plan.delta = J.delta;
    plan.n_pause = 0;
    {
        int idx[TM_MAXNB] = {0};
        for (;;) {
            int best = -1, v = 0;
            for (int b = 0; b < nb; b++) {
                if (sc[b].n_ru > CG_MAX_PAUSES) plan.valid = 0;
                const int n = sc[b].n_ru < CG_MAX_PAUSES ? sc[b].n_ru : CG_MAX_PAUSES;
                if (idx[b] < n && (best < 0 || sc[b].pause_iter[idx[b]] < v)) { best = b; v = sc[b].pause_iter[idx[b]]; }
            }
            if (best < 0) break;
            idx[best]++;
            if (plan.n_pause && plan.pause_iter[plan.n_pause - 1] == v) continue;
            if (plan.n_pause == CG_MAX_PAUSES) { plan.valid = 0; break; }
            plan.pause_iter[plan.n_pause++] = v;
        }
    }
    float ms = 0;
    cudaEventElapsedTime(&ms, J.e0, J.e1);
    tm_status ret = TM_OK;
    for (int b = 0; b < nb; b++) {
        const double eta2 = sc[b].slot[0];
        const double resid = eta2 > 0 ? sqrt(sc[b].rr_true / eta2) : 0.0;
        if (info) {
            info[b].iters = sc[b].iters;
            info[b].reliable_updates = sc[b].n_ru;
            info[b].true_resid = resid;
            info[b].ms = ms / nb;
        }
        if (sc[b].done != 2) {
            snprintf(ctx->err, sizeof(ctx->err), "solve: rho = %g not reached in %d iterations (true residual %g)",
                     P->rho, sc[b].iters, resid);
            ret = TM_ENOCONV;
        }
    }
    return ret;
}

tm_status tm_solve_internal(tm_ctx* ctx, void* d_s, const void* d_eta, double kappa, double mu,
                            const tm_solve_params* P, tm_solve_info* info, cudaStream_t st) {
    SolveJob J;
    TM_TRY(tm_solve_begin(ctx, &J, d_s, d_eta, kappa, mu, P, st, 0.0, 1));
    return tm_solve_end(ctx, &J, info);
}

extern "C" tm_status tm_cg_solve(tm_ctx* ctx, void* d_s, const void* d_eta, double kappa, double mu,
                                 const tm_solve_params* params, tm_solve_info* info, void* stream) {
    if (!ctx || !d_s || !d_eta || !params) return tm_fail(ctx, TM_EARG, "tm_cg_solve: null argument");
    cudaStream_t st = (cudaStream_t)stream;
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    const tm_prec po = params->outer;
    if (po != TM_F64 && po != TM_F32) return tm_fail(ctx, TM_EPREC, "tm_cg_solve: outer precision must be f32 or f64");
    void *eta_i, *s_i;
    TM_TRY(tm_ws(ctx, WS_OU_ETA, 2 * tm_parity_bytes(ctx, po), &eta_i));
    TM_TRY(tm_ws(ctx, WS_OU_S, 2 * tm_parity_bytes(ctx, po), &s_i));
    TM_TRY(tm_import_launch(ctx, eta_i, d_eta, po, st));
    tm_status s = tm_solve_internal(ctx, s_i, eta_i, kappa, mu, params, info, st);
    if (s != TM_OK && s != TM_ENOCONV) return s;
    TM_TRY(tm_export_launch(ctx, d_s, s_i, po, st));
    TM_CUDA(ctx, cudaStreamSynchronize(st));
    return s;
}
