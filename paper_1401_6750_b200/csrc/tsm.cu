// tsm.cu -- Truncated Solver Method estimator loop (sec 2.1) and the
// binary storage of partial sums (sec 2.1.1, Fig. 2; row f2).
//
//   L_TSM = (1/N_LP) sum_{r<N_LP} l_r^LP + (1/N_HP) sum_{r<N_HP} (l_r^HP - l_r^LP)
// with the HP sources = the first N_HP of the LP sources (reading 14).  Per (source, pass) job:
// Z4 noise expanded on the device -> solve (LP, and HP for r < N_HP) -> fused contraction + projection ->
// momentum-space accumulators S_LP, S_LPc, S_HP (device, complex128).  TM_NLANES jobs are in flight at a
// time, each on its own lane (private workspaces, CG state and stream; common.cuh), so that the draining
// tail and the launch gap of every kernel are covered by another source's kernels.  Nothing crosses to the
// host per source except the solver's convergence scalars (and, in tsm_estimate_host, the packed noise).
#include <math.h>
#include <vector>
#include <stdlib.h>
#include "kernels.h"

// acc0 += x ; acc1 += x (optional) ; copy = x (optional)
__global__ void tsm_accumulate_kernel(double* __restrict__ acc0, double* __restrict__ acc1,
                                      double* __restrict__ copy, const double* __restrict__ x, size_t n) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double v = x[i];
    acc0[i] += v;
    if (acc1) acc1[i] += v;
    if (copy) copy[i] = v;
}

// out = S_LP / n_lp + (S_HP - S_LPc) / n_hp, the three sums taken over the lanes in lane order
// (raw != 0: out[3][n] = the three sums themselves, for the all-reduce of a multi-GPU run: SURVEY.md sec 8e)
struct TsmLaneAcc { int n; const double* acc[TM_NLANES]; };
__global__ void tsm_combine_kernel(double* __restrict__ out, TsmLaneAcc L, double inv_lp, double inv_hp, size_t n, int raw) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double slp = 0.0, slpc = 0.0, shp = 0.0;
    for (int l = 0; l < L.n; l++) {
        slp += L.acc[l][i]; slpc += L.acc[l][n + i]; shp += L.acc[l][2 * n + i];
    }
    if (raw) { out[i] = slp; out[n + i] = slpc; out[2 * n + i] = shp; }
    else out[i] = slp * inv_lp + (shp - slpc) * inv_hp;
}
// out = S_LP / n_lp + (S_HP - S_LPc) / n_hp from the raw sums [3][n] (after the all-reduce over ranks)
__global__ void tsm_combine_sums_kernel(double* __restrict__ out, const double* __restrict__ sums, double inv_lp,
                                        double inv_hp, size_t n) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    out[i] = sums[i] * inv_lp + (sums[2 * n + i] - sums[n + i]) * inv_hp;
}

// binary storage (sec 2.1.1): file += x  |  file += x - y
__global__ void binary_add_kernel(double* __restrict__ file, const double* __restrict__ x,
                                  const double* __restrict__ y, size_t n) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    file[i] += y ? x[i] - y[i] : x[i];
}
// out = (sum of the files whose bit is set in mask) / N, summed in ascending file order
__global__ void binary_recover_kernel(double* __restrict__ out, const double* __restrict__ files, unsigned mask,
                                      double inv_n, size_t n) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double s = 0.0;
    for (int k = 0; k < 32; k++)
        if ((mask >> k) & 1u) s += files[(size_t)k * n + i];
    out[i] = s * inv_n;
}

static inline int binary_file_of(int r) {       // 2^k - 1 <= r < 2^(k+1) - 1
    int k = 0;
    while (((1L << (k + 1)) - 1) <= r) k++;
    return k;
}

extern "C" int loop_binary_nfiles(int n_sources) {
    int k = 0;
    while (((1L << k) - 1) < n_sources) k++;
    return k;
}

extern "C" tm_status loop_binary_accumulate(tm_ctx* ctx, void* d_files, const void* d_loop, int r, size_t len,
                                            void* stream) {
    if (!ctx || !d_files || !d_loop || r < 0 || len == 0) return tm_fail(ctx, TM_EARG, "loop_binary_accumulate: bad argument");
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t nr = 2 * len;
    binary_add_kernel<<<(unsigned)((nr + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
        (double*)d_files + (size_t)binary_file_of(r) * nr, (const double*)d_loop, nullptr, nr);
    TM_LAUNCH_CHECK(ctx, "binary_add_kernel");
    return TM_OK;
}

extern "C" tm_status loop_binary_recover(tm_ctx* ctx, void* d_out, const void* d_files, int n_stored, int N,
                                         size_t len, void* stream) {
    if (!ctx || !d_out || !d_files || len == 0) return tm_fail(ctx, TM_EARG, "loop_binary_recover: bad argument");
    if (N < 1 || N > n_stored) return tm_fail(ctx, TM_EARG, "loop_binary_recover: need 1 <= N <= n_stored");
    // "one can recover the data for any number of sources": N = n_stored is the sum of EVERY file, the
    // partially filled last one included; any other N must be made of complete files (file k is complete when all of
    // its 2^k sources are in: 2^(k+1) - 1 <= n_stored), named by its binary digits
    unsigned mask = (unsigned)N;
    if (N == n_stored) mask = (1u << loop_binary_nfiles(n_stored)) - 1u;
    else
        for (int k = 0; (1L << k) <= N; k++)
            if (((N >> k) & 1) && ((1L << (k + 1)) - 1) > n_stored)
                return tm_fail(ctx, TM_EARG, "loop_binary_recover: N needs a file that is not complete yet");
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t nr = 2 * len;
    binary_recover_kernel<<<(unsigned)((nr + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
        (double*)d_out, (const double*)d_files, mask, 1.0 / N, nr);
    TM_LAUNCH_CHECK(ctx, "binary_recover_kernel");
    return TM_OK;
}

// full-lattice field precision conversion (two parity blocks)
static tm_status convert_full(tm_ctx* ctx, void* dst, tm_prec pd, const void* src, tm_prec ps, cudaStream_t st) {
    for (int p = 0; p < 2; p++)
        TM_TRY(blas_copy(ctx, (char*)dst + p * tm_parity_bytes(ctx, pd), pd,
                         (const char*)src + p * tm_parity_bytes(ctx, ps), ps, st));
    return TM_OK;
}

// one unit of work in flight on a lane: the same pass (LP | HP) of nb = 1, 2, 4 or 8 consecutive sources, solved together
struct TsmJob {
    int r, nb, pass;
    SolveJob sj;
    void *eta_o, *s_o;          // nb full-lattice fields back to back, outer precision of the pass
    tm_prec po, ac;
    cudaStream_t st;
};

#ifndef TM_GROUP_DEFAULT
#define TM_GROUP_DEFAULT 8
#endif

struct TsmRun {
    tm_ctx* ctx; const tsm_params* P; void* d_per_source; void* d_files_lp; void* d_files_corr;
    const unsigned char* z4; int z4_on_host; int raw_sums;
    long src_first, src_stride;       // local source j is global source src_first + j * src_stride (its noise stream)
    size_t nr, z4_bytes; unsigned agrid;
    double ms_lp, ms_hp, worst_lp, worst_hp; long it_lp, it_hp; int noconv;
    double* acc[TM_NLANES];         // per lane: S_lp, S_lpc, S_hp, tmp (nr doubles each)
    int group;                      // sources per solve (1 | 2 | 4 | 8; TM_OPT_GROUP, default TM_GROUP_DEFAULT)
    double* lp_keep;                // [TM_MAXNB][nr]: l^LP of the pair whose HP pass comes next (binary files of the correction)
    // host noise (tsm_estimate_host): the whole packed noise of the run is prefetched into one device buffer on the
    // context's copy stream, one chunk (= one group of sources) and one event at a time, while earlier groups solve
    unsigned char* z4_all;          // device [n_lp][3V] (NULL: per-source staging on the lane's own stream)
    std::vector<cudaEvent_t>* z4_ev;    // event of chunk k = sources [k * group, (k + 1) * group)
};

// lane-private buffers of the active lane
static tm_status lane_buffers(TsmRun& R, int lane, cudaStream_t st) {
    tm_ctx* ctx = R.ctx;
    if (R.acc[lane]) return TM_OK;
    TM_TRY(tm_ws(ctx, WS_TSM_ACC, 4 * R.nr * sizeof(double), (void**)&R.acc[lane]));
    TM_CUDA(ctx, cudaMemsetAsync(R.acc[lane], 0, 3 * R.nr * sizeof(double), st));
    return TM_OK;
}

// noise of source r in precision p into slot b of the active lane's (TM_MAXNB-field) buffer
static tm_status job_noise(TsmRun& R, int r, int b, tm_prec p, cudaStream_t st, void** base) {
    tm_ctx* ctx = R.ctx;
    const unsigned char* zsrc = nullptr;
    if (R.z4) {
        if (R.z4_on_host && R.z4_all) {
            TM_CUDA(ctx, cudaStreamWaitEvent(st, (*R.z4_ev)[r / R.group], 0));
            zsrc = R.z4_all + (size_t)r * R.z4_bytes;
        } else if (R.z4_on_host) {
            // staged per lane and slot: the previous user of the slot (a z4_expand of this lane) finished before
            // that lane's solve was waited for
            void* slot;
            TM_TRY(tm_ws(ctx, WS_TSM_Z4, TM_MAXNB * R.z4_bytes, &slot));
            slot = (char*)slot + (size_t)b * R.z4_bytes;
            TM_CUDA(ctx, cudaMemcpyAsync(slot, R.z4 + (size_t)r * R.z4_bytes, R.z4_bytes, cudaMemcpyHostToDevice, st));
            zsrc = (const unsigned char*)slot;
        } else zsrc = R.z4 + (size_t)r * R.z4_bytes;
    }
    const size_t fb = 2 * tm_parity_bytes(ctx, p);
    TM_TRY(tm_ws(ctx, p == TM_F32 ? WS_TSM_ETA32 : WS_TSM_ETA64, TM_MAXNB * fb, base));
    return tm_z4_expand(ctx, (char*)*base + (size_t)b * fb, p, zsrc, R.P->seed,
                        (unsigned long long)(R.src_first + (long)r * R.src_stride), st);
}

static tm_status job_start(TsmRun& R, TsmJob& J, int r, int nb, int pass, cudaStream_t st) {
    tm_ctx* ctx = R.ctx;
    const tsm_params* P = R.P;
    J.r = r; J.nb = nb; J.pass = pass; J.st = st;
    J.po = pass ? P->hp.outer : P->lp.outer;
    J.ac = pass ? P->contract_acc_hp : P->contract_acc_lp;
    for (int b = 0; b < nb; b++) TM_TRY(job_noise(R, r + b, b, J.po, st, &J.eta_o));
    TM_TRY(tm_ws(ctx, J.po == TM_F32 ? WS_TSM_S32 : WS_TSM_S64, TM_MAXNB * 2 * tm_parity_bytes(ctx, J.po), &J.s_o));
    // Z4 noise: |eta_c| = 1 for each of the 12 V components, so ||eta||^2 = 12 V exactly (no norm kernel)
    return tm_solve_begin(ctx, &J.sj, J.s_o, J.eta_o, P->kappa, P->mu, pass ? &P->hp : &P->lp, st, 12.0 * (double)ctx->V, nb);
}

static tm_status job_finish(TsmRun& R, TsmJob& J, int lane) {
    tm_ctx* ctx = R.ctx;
    const tsm_params* P = R.P;
    cudaStream_t st = J.st;
    tm_solve_info si[TM_MAXNB];
    tm_status s = tm_solve_end(ctx, &J.sj, si);
    if (s != TM_OK && s != TM_ENOCONV) return s;
    double* A = R.acc[lane];
    const size_t nr = R.nr;
    double *S_lp = A, *S_lpc = A + nr, *S_hp = A + 2 * nr, *tmp = A + 3 * nr;
    // Merged LP groups: the z-sum, the assembly and the accumulation are linear in the x/y partial sums of the
    // contraction, so the sources of a group whose loops are only ever added into S_LP (no HP partner, no per-source
    // output, no binary files) add their partial sums in the contraction's workspace and share ONE z-sum + assembly +
    // accumulation (fp32 sums of at most 8 sources: inside the fp32-accumulate contract of the LP contraction).
    const bool merged = !J.pass && J.nb > 1 && J.r >= P->n_hp && !R.d_per_source && !R.d_files_lp && !R.lp_keep
                        && J.ac == J.po && tm_contract_merge_ok(ctx, J.ac);
    for (int b = 0; b < J.nb; b++) {
        const int r = J.r + b;
        if (J.pass) { R.ms_hp += si[b].ms; R.it_hp += si[b].iters; R.worst_hp = fmax(R.worst_hp, si[b].true_resid); }
        else        { R.ms_lp += si[b].ms; R.it_lp += si[b].iters; R.worst_lp = fmax(R.worst_lp, si[b].true_resid); }
        const tm_solve_params* sp = J.pass ? &P->hp : &P->lp;
        if (!(si[b].true_resid <= sp->rho * (1.0 + 1e-12))) R.noconv++;
        const size_t fbo = 2 * tm_parity_bytes(ctx, J.po);
        void *s_c = (char*)J.s_o + b * fbo, *eta_c = (char*)J.eta_o + b * fbo;
        if (P->d_solutions)      // the run's own solution of this (source, pass), canonical layout, for the checker
            TM_TRY(tm_export_launch(ctx, (char*)P->d_solutions + (size_t)(J.pass ? P->n_lp + r : r) * ctx->V * 12 * 16,
                                    s_c, J.po, st));
        if (J.ac != J.po) {
            const size_t fba = 2 * tm_parity_bytes(ctx, J.ac);
            void* sbuf;
            TM_TRY(tm_ws(ctx, J.ac == TM_F32 ? WS_TSM_S32 : WS_TSM_S64, TM_MAXNB * fba, &sbuf));
            TM_TRY(convert_full(ctx, sbuf, J.ac, s_c, J.po, st));
            s_c = sbuf;
            void* ebase;
            TM_TRY(job_noise(R, r, 0, J.ac, st, &ebase));
            eta_c = ebase;
        }
        if (merged) {
            const int last = b == J.nb - 1;
            TM_TRY(tm_contract_internal(ctx, tmp, s_c, eta_c, P->kappa, P->mu, P->h_momenta, P->nmom, J.ac, st, 0, 0,
                                        (b > 0 ? 1 : 0) | (last ? 0 : 2)));
            if (!last) continue;
            tsm_accumulate_kernel<<<R.agrid, 256, 0, st>>>(S_lp, nullptr, nullptr, tmp, nr);      // the group's sum
            TM_LAUNCH_CHECK(ctx, "tsm_accumulate_kernel");
            continue;
        }
        TM_TRY(tm_contract_internal(ctx, tmp, s_c, eta_c, P->kappa, P->mu, P->h_momenta, P->nmom, J.ac, st));
        const int do_hp = r < P->n_hp;
        double* copy = R.d_per_source ? (double*)R.d_per_source + (size_t)(J.pass ? P->n_lp + r : r) * nr : nullptr;
        if (J.pass) tsm_accumulate_kernel<<<R.agrid, 256, 0, st>>>(S_hp, nullptr, copy, tmp, nr);
        else        tsm_accumulate_kernel<<<R.agrid, 256, 0, st>>>(S_lp, do_hp ? S_lpc : nullptr, copy, tmp, nr);
        TM_LAUNCH_CHECK(ctx, "tsm_accumulate_kernel");
        if (!J.pass && R.d_files_lp) {
            binary_add_kernel<<<R.agrid, 256, 0, st>>>((double*)R.d_files_lp + (size_t)binary_file_of(r) * nr, tmp, nullptr, nr);
            TM_LAUNCH_CHECK(ctx, "binary_add_kernel");
        }
        if (R.lp_keep && do_hp) {
            double* keep = R.lp_keep + (size_t)(r % TM_MAXNB) * nr;
            if (!J.pass) TM_CUDA(ctx, cudaMemcpyAsync(keep, tmp, nr * sizeof(double), cudaMemcpyDeviceToDevice, st));
            else {
                binary_add_kernel<<<R.agrid, 256, 0, st>>>((double*)R.d_files_corr + (size_t)binary_file_of(r) * nr, tmp, keep, nr);
                TM_LAUNCH_CHECK(ctx, "binary_add_kernel");
            }
        }
    }
    return TM_OK;
}

// Software pipeline over the (source, pass) jobs: TM_NLANES jobs are in flight, each on its own lane (private
// workspaces, device CG state and stream), so the draining tail and launch gap of every kernel of one source
// are filled by kernels of another.  Lane l accumulates into its own S_lp / S_lpc / S_hp; the lanes are joined
// and summed by the final combine kernel.  Job j runs on lane j % NL: results do not depend on timing.
static tm_status tsm_pipeline(TsmRun& R, int NL, cudaStream_t st, void* d_out) {
    tm_ctx* ctx = R.ctx;
    const tsm_params* P = R.P;
    // everything shared between lanes is built on the caller's stream before the lanes fork
    const void* g;
    TM_TRY(tm_get_gauge(ctx, P->lp.sloppy, P->lp.recon, st, &g));
    TM_TRY(tm_get_gauge(ctx, P->lp.outer, P->lp.recon, st, &g));
    TM_TRY(tm_get_gauge(ctx, P->contract_acc_lp, P->contract_acc_lp == TM_F64 ? TM_R18 : TM_R12, st, &g));
    if (P->n_hp) {
        TM_TRY(tm_get_gauge(ctx, P->hp.sloppy, P->hp.recon, st, &g));
        TM_TRY(tm_get_gauge(ctx, P->hp.outer, P->hp.recon, st, &g));
        TM_TRY(tm_get_gauge(ctx, P->contract_acc_hp, P->contract_acc_hp == TM_F64 ? TM_R18 : TM_R12, st, &g));
    }
    cudaEvent_t fork = ctx->ev[5];                 // lane 0's
    TM_CUDA(ctx, cudaEventRecord(fork, st));
    cudaStream_t lst[TM_NLANES];
    for (int l = 0; l < NL; l++) {
        TM_TRY(tm_lane_use(ctx, l));
        lst[l] = l ? ctx->lane_stream : st;
        if (l) TM_CUDA(ctx, cudaStreamWaitEvent(lst[l], fork, 0));
        TM_TRY(lane_buffers(R, l, lst[l]));
    }
    // job list: sources in groups of R.group; a group's LP pass (split into solves of 4, 2 or 1 sources) is followed
    // by the HP pass of those of its sources that have one (r < n_hp)
    struct JobSpec { int r, nb, pass; };
    std::vector<JobSpec> list;
    for (int g = 0; g < P->n_lp; g += R.group)
        for (int pass = 0; pass < 2; pass++) {
            const int lim = pass ? P->n_hp : P->n_lp;
            int r = g, m = lim - g < R.group ? lim - g : R.group;
            while (m > 0) {
                int nb = 1;
                while (2 * nb <= m && 2 * nb <= TM_MAXNB) nb *= 2;
                list.push_back({r, nb, pass});
                r += nb; m -= nb;
            }
        }
    TsmJob jobs[TM_NLANES];
    bool busy[TM_NLANES] = {false};
    const int njobs = (int)list.size();
    for (int j = 0; j < njobs + NL; j++) {
        const int l = j % NL;
        TM_TRY(tm_lane_use(ctx, l));
        if (busy[l]) { TM_TRY(job_finish(R, jobs[l], l)); busy[l] = false; }
        if (j < njobs) {
            TM_TRY(job_start(R, jobs[l], list[j].r, list[j].nb, list[j].pass, lst[l]));
            busy[l] = true;
        }
    }
    // join
    cudaEvent_t joined[TM_NLANES];
    for (int l = 1; l < NL; l++) {
        TM_TRY(tm_lane_use(ctx, l));
        joined[l] = ctx->ev[5];
        TM_CUDA(ctx, cudaEventRecord(joined[l], lst[l]));
    }
    TM_TRY(tm_lane_use(ctx, 0));
    for (int l = 1; l < NL; l++) TM_CUDA(ctx, cudaStreamWaitEvent(st, joined[l], 0));
    TsmLaneAcc LA;
    LA.n = NL;
    for (int l = 0; l < TM_NLANES; l++) LA.acc[l] = l < NL ? R.acc[l] : nullptr;
    tsm_combine_kernel<<<R.agrid, 256, 0, st>>>((double*)d_out, LA, 1.0 / P->n_lp, P->n_hp ? 1.0 / P->n_hp : 0.0, R.nr, R.raw_sums);
    TM_LAUNCH_CHECK(ctx, "tsm_combine_kernel");
    return TM_OK;
}

static tm_status tsm_core(tm_ctx* ctx, void* d_out, void* d_per_source, const tsm_params* P, tsm_info* info,
                          const unsigned char* z4, int z4_on_host, cudaStream_t st,
                          void* d_files_lp = nullptr, void* d_files_corr = nullptr, int raw_sums = 0) {
    if (!P || !d_out) return tm_fail(ctx, TM_EARG, "tsm_estimate: null argument");
    if (P->n_lp < 1 || P->n_hp < 0 || P->n_hp > P->n_lp)
        return tm_fail(ctx, TM_EARG, "tsm_estimate: need 1 <= n_lp and 0 <= n_hp <= n_lp");
    if (P->nmom < 1 || !P->h_momenta) return tm_fail(ctx, TM_EARG, "tsm_estimate: need at least one momentum");
    const tm_prec po_lp = P->lp.outer, po_hp = P->hp.outer;
    const tm_prec ac_lp = P->contract_acc_lp, ac_hp = P->contract_acc_hp;
    if ((po_lp != TM_F32 && po_lp != TM_F64) || (P->n_hp && po_hp != TM_F32 && po_hp != TM_F64))
        return tm_fail(ctx, TM_EPREC, "tsm_estimate: outer precisions must be f32 or f64");
    if ((ac_lp != TM_F32 && ac_lp != TM_F64) || (ac_hp != TM_F32 && ac_hp != TM_F64))
        return tm_fail(ctx, TM_EPREC, "tsm_estimate: contraction precisions must be f32 or f64");
    if ((int)P->lp.sloppy < 0 || (int)P->lp.sloppy > 3 || (int)P->hp.sloppy < 0 || (int)P->hp.sloppy > 3)
        return tm_fail(ctx, TM_EPREC, "tsm_estimate: unknown sloppy precision");
    if ((P->lp.recon != TM_R12 && P->lp.recon != TM_R18) || (P->hp.recon != TM_R12 && P->hp.recon != TM_R18))
        return tm_fail(ctx, TM_EARG, "tsm_estimate: recon must be 12 or 18");
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    TM_TRY(tm_lane_use(ctx, 0));
    const long launches0 = ctx->launches;
    TsmRun R;
    memset(&R, 0, sizeof(R));
    R.ctx = ctx; R.P = P; R.d_per_source = d_per_source; R.d_files_lp = d_files_lp; R.d_files_corr = d_files_corr;
    R.z4 = z4; R.z4_on_host = z4_on_host; R.raw_sums = raw_sums;
    R.src_first = P->src_first; R.src_stride = P->src_stride > 0 ? P->src_stride : 1;
    if (P->src_first < 0 || P->src_stride < 0) return tm_fail(ctx, TM_EARG, "tsm_estimate: src_first and src_stride must be >= 0");
    R.nr = 2 * (size_t)160 * P->nmom * ctx->X[3];                // doubles per per-source array
    R.z4_bytes = 3 * ctx->V;
    R.agrid = (unsigned)((R.nr + 255) / 256);
    {
        // sources per solve: TM_GROUP_DEFAULT, reduced until the lanes' workspaces (noise + solution in outer precision,
        // 5 sloppy vectors, x and r, 3 outer-precision vectors per source; the HP pass is the larger one) stay below
        // 45 % of the device memory, so that a large lattice degrades to smaller groups instead of running out of
        // memory (48^3x96: groups of 4).  tm_set_option(TM_OPT_GROUP) overrides (tuning / tests).
        auto per_source = [&](const tm_solve_params& sp) {
            const double bo = (double)tm_parity_bytes(ctx, sp.outer), bs = (double)tm_parity_bytes(ctx, sp.sloppy);
            const double ba = (double)tm_parity_bytes(ctx, sp.sloppy == TM_F64 ? TM_F64 : TM_F32);
            return 7.0 * bo + 5.0 * bs + 2.0 * ba;
        };
        double need = per_source(P->lp);
        if (P->n_hp && per_source(P->hp) > need) need = per_source(P->hp);
        size_t free_b = 0, total_b = 0;
        TM_CUDA(ctx, cudaMemGetInfo(&free_b, &total_b));
        int gsz = TM_GROUP_DEFAULT;
        while (gsz > 1 && (double)gsz * TM_NLANES * need > 0.45 * (double)total_b) gsz /= 2;
        if (ctx->opt_group) gsz = ctx->opt_group;          // tm_set_option(TM_OPT_GROUP)
        R.group = 1;
        while (2 * R.group <= gsz && 2 * R.group <= TM_MAXNB) R.group *= 2;
    }
    // the binary-storage files are shared accumulators: one lane keeps their additions ordered
    // TM_OPT_LANES, else automatic: kernels that cover 8 sources fill the GPU by themselves, a second job in flight then
    // only adds cache pressure (measured at c4, three A/B pairs on one box: 2089-2129 ms per step on one lane against
    // 2104-2131 ms on two); smaller groups (memory-bound choice, ragged runs) keep two lanes to cover launch gaps
    int NL = ctx->opt_lanes ? ctx->opt_lanes : (R.group >= 8 ? 1 : TM_NLANES);
    if (d_files_lp || d_files_corr || P->n_lp + P->n_hp < 2) NL = 1;
    if (d_files_lp) TM_CUDA(ctx, cudaMemsetAsync(d_files_lp, 0, (size_t)loop_binary_nfiles(P->n_lp) * R.nr * sizeof(double), st));
    if (d_files_corr && P->n_hp) {
        TM_CUDA(ctx, cudaMemsetAsync(d_files_corr, 0, (size_t)loop_binary_nfiles(P->n_hp) * R.nr * sizeof(double), st));
        TM_TRY(tm_ws(ctx, WS_TSM_KEEP, TM_MAXNB * R.nr * sizeof(double), (void**)&R.lp_keep));
    }
    cudaEvent_t e0 = ctx->ev[2], e1 = ctx->ev[3];
    TM_CUDA(ctx, cudaEventRecord(e0, st));
    std::vector<cudaEvent_t> z4_events;
    if (z4 && z4_on_host) {
        // 180 GB of HBM: the packed noise of a whole run (3V bytes per source: 3.1 GB for 500 sources at 32^3x64) stays
        // resident.  It is uploaded on the copy stream in group-sized chunks behind the caller's stream (e0), each chunk
        // with its own event, so only the first group's copy is exposed; the lanes wait per chunk (job_noise).  A run whose
        // noise would take more than a quarter of the free memory keeps the per-source staging on the lane's stream.
        size_t free_b = 0, total_b = 0;
        TM_CUDA(ctx, cudaMemGetInfo(&free_b, &total_b));
        const size_t all = (size_t)P->n_lp * R.z4_bytes;
        void* buf = nullptr;
        if (all <= free_b / 4 + ctx->scratch_bytes[WS_TSM_Z4] && tm_ws(ctx, WS_TSM_Z4, all, &buf) == TM_OK) {
            if (!ctx->copy_stream) TM_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
            TM_CUDA(ctx, cudaStreamWaitEvent(ctx->copy_stream, e0, 0));
            R.z4_all = (unsigned char*)buf;
            R.z4_ev = &z4_events;
            for (int r0 = 0; r0 < P->n_lp; r0 += R.group) {
                const int n = P->n_lp - r0 < R.group ? P->n_lp - r0 : R.group;
                TM_CUDA(ctx, cudaMemcpyAsync(R.z4_all + (size_t)r0 * R.z4_bytes, z4 + (size_t)r0 * R.z4_bytes,
                                             (size_t)n * R.z4_bytes, cudaMemcpyHostToDevice, ctx->copy_stream));
                cudaEvent_t ev;
                TM_CUDA(ctx, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
                z4_events.push_back(ev);
                TM_CUDA(ctx, cudaEventRecord(ev, ctx->copy_stream));
            }
        } else cudaGetLastError();
    }
    tm_status s = tsm_pipeline(R, NL, st, d_out);
    if (!z4_events.empty()) {
        if (s != TM_OK) cudaStreamSynchronize(ctx->copy_stream);
        for (cudaEvent_t ev : z4_events) cudaEventDestroy(ev);     // deferred by the runtime until the event has completed
    }
    if (s != TM_OK) {
        // leave no lane running behind the caller's back
        for (int l = 1; l < NL; l++)
            if (tm_lane_use(ctx, l) == TM_OK && ctx->lane_stream) cudaStreamSynchronize(ctx->lane_stream);
        char keep[sizeof(ctx->err)];
        memcpy(keep, ctx->err, sizeof(keep));
        tm_lane_use(ctx, 0);
        memcpy(ctx->err, keep, sizeof(keep));
        cudaGetLastError();
        return s;
    }
    TM_CUDA(ctx, cudaEventRecord(e1, st));
    TM_CUDA(ctx, cudaEventSynchronize(e1));
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (info) {
        // with NL solves in flight the per-solve elapsed times overlap: their sums are divided by NL
        info->ms_total = ms; info->ms_lp_solve = R.ms_lp / NL; info->ms_hp_solve = R.ms_hp / NL;
        info->ms_contract = ms - info->ms_lp_solve - info->ms_hp_solve;   // contraction + noise expansion + accumulation
        info->iters_lp = R.it_lp; info->iters_hp = R.it_hp;
        info->worst_resid_lp = R.worst_lp; info->worst_resid_hp = R.worst_hp;
        info->launches = (int)(ctx->launches - launches0);
        info->lanes = NL;
    }
    if (R.noconv) {
        snprintf(ctx->err, sizeof(ctx->err), "tsm_estimate: %d solve(s) missed their rho (worst LP %g, HP %g)",
                 R.noconv, R.worst_lp, R.worst_hp);
        return TM_ENOCONV;
    }
    return TM_OK;
}

extern "C" tm_status tsm_estimate(tm_ctx* ctx, void* d_out, void* d_per_source, const tsm_params* P,
                                  tsm_info* info, void* stream) {
    if (!ctx) return TM_EARG;
    return tsm_core(ctx, d_out, d_per_source, P, info, P ? P->d_z4 : nullptr, 0, (cudaStream_t)stream);
}

extern "C" tm_status tsm_partial_sums(tm_ctx* ctx, void* d_sums, void* d_per_source, const tsm_params* P,
                                      tsm_info* info, void* stream) {
    if (!ctx) return TM_EARG;
    return tsm_core(ctx, d_sums, d_per_source, P, info, P ? P->d_z4 : nullptr, 0, (cudaStream_t)stream, nullptr, nullptr, 1);
}

extern "C" tm_status tsm_combine_sums(tm_ctx* ctx, void* d_out, const void* d_sums, int n_lp_total, int n_hp_total,
                                      int nmom, void* stream) {
    if (!ctx) return TM_EARG;
    if (!d_out || !d_sums || n_lp_total < 1 || n_hp_total < 0 || nmom < 1)
        return tm_fail(ctx, TM_EARG, "tsm_combine_sums: bad argument");
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t nr = 2 * (size_t)160 * nmom * ctx->X[3];
    tsm_combine_sums_kernel<<<(unsigned)((nr + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
        (double*)d_out, (const double*)d_sums, 1.0 / n_lp_total, n_hp_total ? 1.0 / n_hp_total : 0.0, nr);
    TM_LAUNCH_CHECK(ctx, "tsm_combine_sums_kernel");
    return TM_OK;
}

extern "C" tm_status tsm_estimate_binary(tm_ctx* ctx, void* d_out, void* d_files_lp, void* d_files_corr,
                                         const tsm_params* P, tsm_info* info, void* stream) {
    if (!ctx) return TM_EARG;
    return tsm_core(ctx, d_out, nullptr, P, info, P ? P->d_z4 : nullptr, 0, (cudaStream_t)stream, d_files_lp, d_files_corr);
}

static tm_status tsm_host(tm_ctx* ctx, void* h_out, const unsigned char* h_z4, const tsm_params* P, tsm_info* info,
                          cudaStream_t st, int raw_sums) {
    if (!h_out || !P) return tm_fail(ctx, TM_EARG, "tsm_estimate_host: null argument");
    if (P->nmom < 1) return tm_fail(ctx, TM_EARG, "tsm_estimate_host: need at least one momentum");
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t bytes = (size_t)(raw_sums ? 3 : 1) * 160 * P->nmom * ctx->X[3] * 16;
    void* d_out;
    TM_TRY(tm_ws(ctx, WS_API_B, bytes, &d_out));
    tm_status s = tsm_core(ctx, d_out, nullptr, P, info, h_z4, 1, st, nullptr, nullptr, raw_sums);
    if (s != TM_OK && s != TM_ENOCONV) return s;
    TM_CUDA(ctx, cudaMemcpyAsync(h_out, d_out, bytes, cudaMemcpyDeviceToHost, st));
    TM_CUDA(ctx, cudaStreamSynchronize(st));
    return s;
}

extern "C" tm_status tsm_estimate_host(tm_ctx* ctx, void* h_out, const unsigned char* h_z4, const tsm_params* P,
                                       tsm_info* info, void* stream) {
    if (!ctx) return TM_EARG;
    return tsm_host(ctx, h_out, h_z4, P, info, (cudaStream_t)stream, 0);
}

extern "C" tm_status tsm_partial_sums_host(tm_ctx* ctx, void* h_sums, const unsigned char* h_z4, const tsm_params* P,
                                           tsm_info* info, void* stream) {
    if (!ctx) return TM_EARG;
    return tsm_host(ctx, h_sums, h_z4, P, info, (cudaStream_t)stream, 1);
}
