// tsm.cu -- Truncated Solver Method estimator loop (sec 2.1).
//
//   L_TSM = (1/N_LP) sum_{r<N_LP} l_r^LP + (1/N_HP) sum_{r<N_HP} (l_r^HP - l_r^LP)
// with the HP sources = the first N_HP of the LP sources (reading 14).  Per source:
// Z4 noise expanded on the device -> tm_solve_internal (LP, and HP for r < N_HP) -> fused
// contraction + projection -> momentum-space accumulators S_LP, S_LPc, S_HP (device, complex128).
// Nothing crosses to the host per source except the solver's convergence scalars (and, in
// tsm_estimate_host, the packed noise of that source).
#include <math.h>
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

// out = S_LP / n_lp + (S_HP - S_LPc) / n_hp
__global__ void tsm_combine_kernel(double* __restrict__ out, const double* __restrict__ slp,
                                   const double* __restrict__ slpc, const double* __restrict__ shp,
                                   double inv_lp, double inv_hp, size_t n) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    out[i] = slp[i] * inv_lp + (shp[i] - slpc[i]) * inv_hp;
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
    // file k is complete when all of its 2^k sources are in: 2^(k+1) - 1 <= n_stored
    for (int k = 0; (1L << k) <= N; k++)
        if (((N >> k) & 1) && ((1L << (k + 1)) - 1) > n_stored)
            return tm_fail(ctx, TM_EARG, "loop_binary_recover: N needs a file that is not complete yet");
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t nr = 2 * len;
    binary_recover_kernel<<<(unsigned)((nr + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
        (double*)d_out, (const double*)d_files, (unsigned)N, 1.0 / N, nr);
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

static tm_status tsm_core(tm_ctx* ctx, void* d_out, void* d_per_source, const tsm_params* P, tsm_info* info,
                          const unsigned char* z4, int z4_on_host, cudaStream_t st,
                          void* d_files_lp = nullptr, void* d_files_corr = nullptr) {
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
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    const long launches0 = ctx->launches;
    const size_t nout = (size_t)160 * P->nmom * ctx->X[3];       // complex entries
    const size_t nr = 2 * nout;                                  // doubles
    const size_t z4_bytes = 3 * ctx->V;
    double* acc;
    TM_TRY(tm_ws(ctx, WS_TSM_ACC, 4 * nr * sizeof(double), (void**)&acc));
    double *S_lp = acc, *S_lpc = acc + nr, *S_hp = acc + 2 * nr, *tmp = acc + 3 * nr;
    TM_CUDA(ctx, cudaMemsetAsync(acc, 0, 3 * nr * sizeof(double), st));
    double* lp_keep = nullptr;          // l_r^LP kept until l_r^HP is known (binary files of the correction)
    if (d_files_lp) TM_CUDA(ctx, cudaMemsetAsync(d_files_lp, 0, (size_t)loop_binary_nfiles(P->n_lp) * nr * sizeof(double), st));
    if (d_files_corr && P->n_hp) {
        TM_CUDA(ctx, cudaMemsetAsync(d_files_corr, 0, (size_t)loop_binary_nfiles(P->n_hp) * nr * sizeof(double), st));
        TM_TRY(tm_ws(ctx, WS_TSM_KEEP, nr * sizeof(double), (void**)&lp_keep));
    }
    void *eta32 = nullptr, *eta64 = nullptr, *s32 = nullptr, *s64 = nullptr, *z4dev = nullptr;
    const bool need32 = po_lp == TM_F32 || ac_lp == TM_F32 || (P->n_hp && (po_hp == TM_F32 || ac_hp == TM_F32));
    const bool need64 = po_lp == TM_F64 || ac_lp == TM_F64 || (P->n_hp && (po_hp == TM_F64 || ac_hp == TM_F64));
    if (need32) {
        TM_TRY(tm_ws(ctx, WS_TSM_ETA32, 2 * tm_parity_bytes(ctx, TM_F32), &eta32));
        TM_TRY(tm_ws(ctx, WS_TSM_S32, 2 * tm_parity_bytes(ctx, TM_F32), &s32));
    }
    if (need64) {
        TM_TRY(tm_ws(ctx, WS_TSM_ETA64, 2 * tm_parity_bytes(ctx, TM_F64), &eta64));
        TM_TRY(tm_ws(ctx, WS_TSM_S64, 2 * tm_parity_bytes(ctx, TM_F64), &s64));
    }
    if (z4 && z4_on_host) TM_TRY(tm_ws(ctx, WS_TSM_Z4, 2 * z4_bytes, &z4dev));

    cudaEvent_t e0 = ctx->ev[2], e1 = ctx->ev[3];
    TM_CUDA(ctx, cudaEventRecord(e0, st));
    double ms_lp = 0, ms_hp = 0;
    long it_lp = 0, it_hp = 0;
    double worst_lp = 0, worst_hp = 0;
    int noconv = 0;
    const unsigned agrid = (unsigned)((nr + 255) / 256);

    for (int r = 0; r < P->n_lp; r++) {
        const unsigned char* zsrc = nullptr;
        if (z4) {
            if (z4_on_host) {
                // double-buffered staging: the copy of source r is stream-ordered behind the work of r-1
                unsigned char* slot = (unsigned char*)z4dev + (size_t)(r & 1) * z4_bytes;
                TM_CUDA(ctx, cudaMemcpyAsync(slot, z4 + (size_t)r * z4_bytes, z4_bytes, cudaMemcpyHostToDevice, st));
                zsrc = slot;
            } else zsrc = z4 + (size_t)r * z4_bytes;
        }
        const int do_hp = r < P->n_hp;
        // noise in every precision this source needs
        bool have32 = false, have64 = false;
        auto eta_in = [&](tm_prec p, void** out) -> tm_status {
            if (p == TM_F32) {
                if (!have32) { TM_TRY(tm_z4_expand(ctx, eta32, TM_F32, zsrc, P->seed, (unsigned long long)r, st)); have32 = true; }
                *out = eta32;
            } else {
                if (!have64) { TM_TRY(tm_z4_expand(ctx, eta64, TM_F64, zsrc, P->seed, (unsigned long long)r, st)); have64 = true; }
                *out = eta64;
            }
            return TM_OK;
        };
        for (int pass = 0; pass < 1 + do_hp; pass++) {
            const tm_solve_params* sp = pass ? &P->hp : &P->lp;
            const tm_prec po = pass ? po_hp : po_lp, ac = pass ? ac_hp : ac_lp;
            void *eta_o, *eta_c, *s_o = po == TM_F32 ? s32 : s64, *s_c;
            TM_TRY(eta_in(po, &eta_o));
            tm_solve_info si;
            tm_status s = tm_solve_internal(ctx, s_o, eta_o, P->kappa, P->mu, sp, &si, st);
            if (s == TM_ENOCONV) noconv++;
            else if (s != TM_OK) return s;
            if (pass) { ms_hp += si.ms; it_hp += si.iters; worst_hp = fmax(worst_hp, si.true_resid); }
            else      { ms_lp += si.ms; it_lp += si.iters; worst_lp = fmax(worst_lp, si.true_resid); }
            if (ac == po) { s_c = s_o; eta_c = eta_o; }
            else {
                s_c = ac == TM_F32 ? s32 : s64;
                TM_TRY(convert_full(ctx, s_c, ac, s_o, po, st));
                TM_TRY(eta_in(ac, &eta_c));
            }
            TM_TRY(tm_contract_internal(ctx, tmp, s_c, eta_c, P->kappa, P->mu, P->h_momenta, P->nmom, ac, st));
            double* copy = d_per_source ? (double*)d_per_source + (size_t)(pass ? P->n_lp + r : r) * nr : nullptr;
            if (pass) tsm_accumulate_kernel<<<agrid, 256, 0, st>>>(S_hp, nullptr, copy, tmp, nr);
            else      tsm_accumulate_kernel<<<agrid, 256, 0, st>>>(S_lp, do_hp ? S_lpc : nullptr, copy, tmp, nr);
            TM_LAUNCH_CHECK(ctx, "tsm_accumulate_kernel");
            if (!pass && d_files_lp) {
                binary_add_kernel<<<agrid, 256, 0, st>>>((double*)d_files_lp + (size_t)binary_file_of(r) * nr, tmp, nullptr, nr);
                TM_LAUNCH_CHECK(ctx, "binary_add_kernel");
            }
            if (lp_keep && do_hp) {
                if (!pass) TM_CUDA(ctx, cudaMemcpyAsync(lp_keep, tmp, nr * sizeof(double), cudaMemcpyDeviceToDevice, st));
                else {
                    binary_add_kernel<<<agrid, 256, 0, st>>>((double*)d_files_corr + (size_t)binary_file_of(r) * nr, tmp, lp_keep, nr);
                    TM_LAUNCH_CHECK(ctx, "binary_add_kernel");
                }
            }
        }
    }
    tsm_combine_kernel<<<agrid, 256, 0, st>>>((double*)d_out, S_lp, S_lpc, S_hp, 1.0 / P->n_lp,
                                             P->n_hp ? 1.0 / P->n_hp : 0.0, nr);
    TM_LAUNCH_CHECK(ctx, "tsm_combine_kernel");
    TM_CUDA(ctx, cudaEventRecord(e1, st));
    TM_CUDA(ctx, cudaEventSynchronize(e1));
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (info) {
        info->ms_total = ms; info->ms_lp_solve = ms_lp; info->ms_hp_solve = ms_hp;
        info->ms_contract = ms - ms_lp - ms_hp;      // contraction + noise expansion + accumulation
        info->iters_lp = it_lp; info->iters_hp = it_hp;
        info->worst_resid_lp = worst_lp; info->worst_resid_hp = worst_hp;
        info->launches = (int)(ctx->launches - launches0);
    }
    if (noconv) {
        snprintf(ctx->err, sizeof(ctx->err), "tsm_estimate: %d solve(s) missed their rho (worst LP %g, HP %g)",
                 noconv, worst_lp, worst_hp);
        return TM_ENOCONV;
    }
    return TM_OK;
}

extern "C" tm_status tsm_estimate(tm_ctx* ctx, void* d_out, void* d_per_source, const tsm_params* P,
                                  tsm_info* info, void* stream) {
    if (!ctx) return TM_EARG;
    return tsm_core(ctx, d_out, d_per_source, P, info, P ? P->d_z4 : nullptr, 0, (cudaStream_t)stream);
}

extern "C" tm_status tsm_estimate_binary(tm_ctx* ctx, void* d_out, void* d_files_lp, void* d_files_corr,
                                         const tsm_params* P, tsm_info* info, void* stream) {
    if (!ctx) return TM_EARG;
    return tsm_core(ctx, d_out, nullptr, P, info, P ? P->d_z4 : nullptr, 0, (cudaStream_t)stream, d_files_lp, d_files_corr);
}

extern "C" tm_status tsm_estimate_host(tm_ctx* ctx, void* h_out, const unsigned char* h_z4, const tsm_params* P,
                                       tsm_info* info, void* stream) {
    if (!ctx) return TM_EARG;
    if (!h_out || !P) return tm_fail(ctx, TM_EARG, "tsm_estimate_host: null argument");
    cudaStream_t st = (cudaStream_t)stream;
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t bytes = (size_t)160 * P->nmom * ctx->X[3] * 16;
    void* d_out;
    TM_TRY(tm_ws(ctx, WS_API_B, bytes, &d_out));
    tm_status s = tsm_core(ctx, d_out, nullptr, P, info, h_z4, 1, st);
    if (s != TM_OK && s != TM_ENOCONV) return s;
    TM_CUDA(ctx, cudaMemcpyAsync(h_out, d_out, bytes, cudaMemcpyDeviceToHost, st));
    TM_CUDA(ctx, cudaStreamSynchronize(st));
    return s;
}
