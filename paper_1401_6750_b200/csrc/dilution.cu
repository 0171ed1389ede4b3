// dilution.cu -- time dilution ("we also worked with time-dilution [6], so there are GPU kernels to contract
// a single time slice or a whole vector"; PAPER.md:92 lists it among the variance-reduction methods that combine with
// the TSM; reading 22).
//
// A time-diluted source eta^(t0) is the noise vector restricted to timeslice t0.  With M s^(t0) = eta^(t0) the plain
// stochastic estimator of the loop on that timeslice is
//     l[i][k][t0] = sum_{x in t0} exp(+2 pi i p_k.x / L) eta^(t0)(x)^dag X_i s^(t0)(x),
//     X_n = Gamma_n (n < 16),  X_{16+16m+n} = Gamma_n D_m (D_m on s),
// so one noise vector costs T solves and T single-timeslice contractions, and the noise of the other T-1 timeslices
// never enters.  The bilinear comes out of the 160-insertion primitive of contract.cu launched on ONE timeslice: with
// the pair swapped (s := a, eta := b) and mu = 0 its f = 1 block is a^dag g5 G_n D_m g5 b, and g5 G_n g5 = eps_n G_n
// with eps_n = (-1)^(number of gamma matrices in G_n) because g5 anticommutes with every g_mu.
#include <math.h>
#include <vector>
#include "kernels.h"

// v = eps_n * prim[f = 1][idx] (zero outside column t_only when t_only >= 0);  dst = v | acc0 += v | acc1 += v | copy = v
__global__ void plain_assemble_kernel(double2* __restrict__ dst, double2* __restrict__ acc0, double2* __restrict__ acc1,
                                      double2* __restrict__ copy, const double2* __restrict__ prim, size_t per_f,
                                      int nmom, int T, int t_only) {
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= per_f) return;
    const int i = (int)(idx / ((size_t)nmom * T));
    const int n = i < 16 ? i : (i - 16) & 15;
    const double eps = (__popc(n) & 1) ? -1.0 : 1.0;
    double2 v = prim[per_f + idx];
    v.x *= eps; v.y *= eps;
    if (t_only >= 0 && (int)(idx % T) != t_only) v = make_double2(0.0, 0.0);
    if (dst) dst[idx] = v;
    if (acc0) { double2 a = acc0[idx]; a.x += v.x; a.y += v.y; acc0[idx] = a; }
    if (acc1) { double2 a = acc1[idx]; a.x += v.x; a.y += v.y; acc1[idx] = a; }
    if (copy) copy[idx] = v;
}

// out = S_LP / n_lp + (S_HP - S_LPc) / n_hp on n doubles, sums = [3][n]
__global__ void td_combine_kernel(double* __restrict__ out, const double* __restrict__ sums, double inv_lp, double inv_hp,
                                  size_t n) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    out[i] = sums[i] * inv_lp + (sums[2 * n + i] - sums[n + i]) * inv_hp;
}

extern "C" tm_status loop_plain_project_timeslice(tm_ctx* ctx, void* d_out, const void* d_a, const void* d_b,
                                                  const int* h_momenta, int nmom, int t0, tm_prec acc, void* stream) {
    if (!ctx || !d_out || !d_a || !d_b) return tm_fail(ctx, TM_EARG, "loop_plain_project_timeslice: null argument");
    if (acc != TM_F64 && acc != TM_F32) return tm_fail(ctx, TM_EPREC, "loop_plain_project_timeslice: acc must be f32 or f64");
    if (t0 < -1 || t0 >= ctx->X[3]) return tm_fail(ctx, TM_EARG, "loop_plain_project_timeslice: t0 outside the lattice");
    if (nmom < 1 || !h_momenta) return tm_fail(ctx, TM_EARG, "loop_plain_project_timeslice: need at least one momentum");
    cudaStream_t st = (cudaStream_t)stream;
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t per_f = (size_t)80 * nmom * ctx->X[3];
    void *ai, *bi, *prim;
    TM_TRY(tm_ws(ctx, WS_CT_S, 2 * tm_parity_bytes(ctx, acc), &ai));
    TM_TRY(tm_ws(ctx, WS_CT_ETA, 2 * tm_parity_bytes(ctx, acc), &bi));
    TM_TRY(tm_ws(ctx, WS_API_A, 2 * per_f * 16, &prim));
    TM_TRY(tm_import_launch(ctx, ai, d_a, acc, st));
    TM_TRY(tm_import_launch(ctx, bi, d_b, acc, st));
    if (t0 >= 0) TM_TRY(tm_contract_internal(ctx, prim, ai, bi, 0.0, 0.0, h_momenta, nmom, acc, st, t0, 1));
    else         TM_TRY(tm_contract_internal(ctx, prim, ai, bi, 0.0, 0.0, h_momenta, nmom, acc, st));
    plain_assemble_kernel<<<(unsigned)((per_f + 255) / 256), 256, 0, st>>>((double2*)d_out, nullptr, nullptr, nullptr,
                                                                          (const double2*)prim, per_f, nmom, ctx->X[3], t0);
    TM_LAUNCH_CHECK(ctx, "plain_assemble_kernel");
    return TM_OK;
}

// full-lattice field precision conversion (two parity blocks)
static tm_status td_convert_full(tm_ctx* ctx, void* dst, tm_prec pd, const void* src, tm_prec ps, cudaStream_t st) {
    for (int p = 0; p < 2; p++)
        TM_TRY(blas_copy(ctx, (char*)dst + p * tm_parity_bytes(ctx, pd), pd,
                         (const char*)src + p * tm_parity_bytes(ctx, ps), ps, st));
    return TM_OK;
}

extern "C" tm_status tsm_estimate_time_diluted(tm_ctx* ctx, void* d_out, void* d_per_source, const tsm_params* P,
                                               tsm_info* info, void* stream) {
    if (!ctx) return TM_EARG;
    if (!P || !d_out) return tm_fail(ctx, TM_EARG, "tsm_estimate_time_diluted: null argument");
    if (P->n_lp < 1 || P->n_hp < 0 || P->n_hp > P->n_lp)
        return tm_fail(ctx, TM_EARG, "tsm_estimate_time_diluted: need 1 <= n_lp and 0 <= n_hp <= n_lp");
    if (P->nmom < 1 || !P->h_momenta) return tm_fail(ctx, TM_EARG, "tsm_estimate_time_diluted: need at least one momentum");
    if (P->src_first < 0 || P->src_stride < 0) return tm_fail(ctx, TM_EARG, "tsm_estimate_time_diluted: src_first and src_stride must be >= 0");
    for (int pass = 0; pass < (P->n_hp ? 2 : 1); pass++) {
        const tm_prec po = pass ? P->hp.outer : P->lp.outer, ac = pass ? P->contract_acc_hp : P->contract_acc_lp;
        if (po != TM_F32 && po != TM_F64) return tm_fail(ctx, TM_EPREC, "tsm_estimate_time_diluted: outer precisions must be f32 or f64");
        if (ac != TM_F32 && ac != TM_F64) return tm_fail(ctx, TM_EPREC, "tsm_estimate_time_diluted: contraction precisions must be f32 or f64");
    }
    cudaStream_t st = (cudaStream_t)stream;
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    TM_TRY(tm_lane_use(ctx, 0));
    const long launches0 = ctx->launches;
    const int T = ctx->X[3];
    const size_t per_f = (size_t)80 * P->nmom * T;            // complex entries of one per-source array
    const size_t nrd = 2 * per_f;                             // doubles
    const unsigned agrid = (unsigned)((per_f + 255) / 256);
    const long stride = P->src_stride > 0 ? P->src_stride : 1;
    int group = ctx->opt_group ? ctx->opt_group : TM_MAXNB;
    // timeslices of one noise vector solved together; the group is halved until the workspaces of a group (noise +
    // solution + 3 outer-precision vectors + 7 sloppy ones per source) stay below 45 % of the device memory
    {
        size_t free_b = 0, total_b = 0;
        TM_CUDA(ctx, cudaMemGetInfo(&free_b, &total_b));
        const tm_solve_params& big = P->n_hp ? P->hp : P->lp;
        const double need = 7.0 * (double)tm_parity_bytes(ctx, big.outer) + 7.0 * (double)tm_parity_bytes(ctx, TM_F32);
        while (!ctx->opt_group && group > 1 && (double)group * need > 0.45 * (double)total_b) group /= 2;
    }
    double *sums, *prim;
    TM_TRY(tm_ws(ctx, WS_TD_ACC, 3 * nrd * sizeof(double), (void**)&sums));
    TM_TRY(tm_ws(ctx, WS_TD_PRIM, 2 * nrd * sizeof(double), (void**)&prim));
    TM_CUDA(ctx, cudaMemsetAsync(sums, 0, 3 * nrd * sizeof(double), st));
    cudaEvent_t e0 = ctx->ev[2], e1 = ctx->ev[3];
    TM_CUDA(ctx, cudaEventRecord(e0, st));
    double ms_lp = 0, ms_hp = 0, worst_lp = 0, worst_hp = 0;
    long it_lp = 0, it_hp = 0;
    int noconv = 0;
    const size_t z4_bytes = 3 * ctx->V;
    for (int r = 0; r < P->n_lp; r++)
        for (int pass = 0; pass < (r < P->n_hp ? 2 : 1); pass++) {
            const tm_solve_params* sp = pass ? &P->hp : &P->lp;
            const tm_prec po = sp->outer, ac = pass ? P->contract_acc_hp : P->contract_acc_lp;
            const size_t fbo = 2 * tm_parity_bytes(ctx, po), fba = 2 * tm_parity_bytes(ctx, ac);
            const unsigned char* zsrc = P->d_z4 ? P->d_z4 + (size_t)r * z4_bytes : nullptr;
            const unsigned long long stream_id = (unsigned long long)(P->src_first + (long)r * stride);
            void *eta_o, *s_o;
            TM_TRY(tm_ws(ctx, po == TM_F32 ? WS_TSM_ETA32 : WS_TSM_ETA64, TM_MAXNB * fbo, &eta_o));
            TM_TRY(tm_ws(ctx, po == TM_F32 ? WS_TSM_S32 : WS_TSM_S64, TM_MAXNB * fbo, &s_o));
            for (int t0 = 0; t0 < T;) {
                int nb = 1;
                while (2 * nb <= T - t0 && 2 * nb <= group && 2 * nb <= TM_MAXNB) nb *= 2;
                for (int b = 0; b < nb; b++)
                    TM_TRY(tm_z4_expand(ctx, (char*)eta_o + (size_t)b * fbo, po, zsrc, P->seed, stream_id, st, t0 + b));
                // |eta_c| = 1 on the 12 V / T components of the timeslice
                SolveJob sj;
                TM_TRY(tm_solve_begin(ctx, &sj, s_o, eta_o, P->kappa, P->mu, sp, st, 12.0 * (double)ctx->V / T, nb));
                tm_solve_info si[TM_MAXNB];
                tm_status s = tm_solve_end(ctx, &sj, si);
                if (s != TM_OK && s != TM_ENOCONV) return s;
                for (int b = 0; b < nb; b++) {
                    if (pass) { ms_hp += si[b].ms; it_hp += si[b].iters; worst_hp = fmax(worst_hp, si[b].true_resid); }
                    else      { ms_lp += si[b].ms; it_lp += si[b].iters; worst_lp = fmax(worst_lp, si[b].true_resid); }
                    if (!(si[b].true_resid <= sp->rho * (1.0 + 1e-12))) noconv++;
                    void *s_c = (char*)s_o + (size_t)b * fbo, *eta_c = (char*)eta_o + (size_t)b * fbo;
                    if (ac != po) {
                        void *sbuf, *ebuf;
                        TM_TRY(tm_ws(ctx, ac == TM_F32 ? WS_TSM_S32 : WS_TSM_S64, TM_MAXNB * fba, &sbuf));
                        TM_TRY(tm_ws(ctx, ac == TM_F32 ? WS_TSM_ETA32 : WS_TSM_ETA64, TM_MAXNB * fba, &ebuf));
                        TM_TRY(td_convert_full(ctx, sbuf, ac, s_c, po, st));
                        TM_TRY(tm_z4_expand(ctx, ebuf, ac, zsrc, P->seed, stream_id, st, t0 + b));
                        s_c = sbuf; eta_c = ebuf;
                    }
                    // column t0 + b of the primitive of the swapped pair (eta^(t0), s^(t0)) at mu = 0
                    TM_TRY(tm_contract_internal(ctx, prim, eta_c, s_c, 0.0, 0.0, P->h_momenta, P->nmom, ac, st, t0 + b, 1));
                }
                t0 += nb;
            }
            // every column of prim now belongs to this (noise vector, pass): l_r = eps_n * prim[1]
            double2* S_lp = (double2*)sums, *S_lpc = S_lp + per_f, *S_hp = S_lp + 2 * per_f;
            double2* copy = d_per_source ? (double2*)d_per_source + (size_t)(pass ? P->n_lp + r : r) * per_f : nullptr;
            if (pass) plain_assemble_kernel<<<agrid, 256, 0, st>>>(nullptr, S_hp, nullptr, copy, (const double2*)prim, per_f, P->nmom, T, -1);
            else      plain_assemble_kernel<<<agrid, 256, 0, st>>>(nullptr, S_lp, r < P->n_hp ? S_lpc : nullptr, copy,
                                                                   (const double2*)prim, per_f, P->nmom, T, -1);
            TM_LAUNCH_CHECK(ctx, "plain_assemble_kernel");
        }
    td_combine_kernel<<<(unsigned)((nrd + 255) / 256), 256, 0, st>>>((double*)d_out, sums, 1.0 / P->n_lp,
                                                                    P->n_hp ? 1.0 / P->n_hp : 0.0, nrd);
    TM_LAUNCH_CHECK(ctx, "td_combine_kernel");
    TM_CUDA(ctx, cudaEventRecord(e1, st));
    TM_CUDA(ctx, cudaEventSynchronize(e1));
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (info) {
        info->ms_total = ms; info->ms_lp_solve = ms_lp; info->ms_hp_solve = ms_hp;
        info->ms_contract = ms - ms_lp - ms_hp;
        info->iters_lp = it_lp; info->iters_hp = it_hp;
        info->worst_resid_lp = worst_lp; info->worst_resid_hp = worst_hp;
        info->launches = (int)(ctx->launches - launches0);
        info->lanes = 1;
    }
    if (noconv) {
        snprintf(ctx->err, sizeof(ctx->err), "tsm_estimate_time_diluted: %d solve(s) missed their rho (worst LP %g, HP %g)",
                 noconv, worst_lp, worst_hp);
        return TM_ENOCONV;
    }
    return TM_OK;
}
