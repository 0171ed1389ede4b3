// api.cu -- context lifetime, workspaces and the exported tm_dslash / field conversion calls.
#include <stdlib.h>
#include "kernels.h"

static char g_last_error[512] = "";

extern "C" const char* tm_last_error(const tm_ctx* ctx) { return ctx ? ctx->err : g_last_error; }
extern "C" long tm_launch_count(const tm_ctx* ctx) { return ctx ? ctx->launches : 0; }

// allocate the private resources of a lane into the context's active fields
static bool lane_alloc(tm_ctx* c, int lane) {
    bool ok = cudaMalloc((void**)&c->d_partials, sizeof(double) * TM_MAXNB * TM_PSTRIDE) == cudaSuccess
           && cudaMalloc((void**)&c->d_counter, sizeof(unsigned int) * TM_MAXNB) == cudaSuccess
           && cudaMalloc((void**)&c->d_scal, TM_MAXNB * sizeof(CgScalars)) == cudaSuccess
           && cudaMallocHost((void**)&c->h_scal, TM_MAXNB * sizeof(CgScalars)) == cudaSuccess
           && cudaMemset(c->d_counter, 0, sizeof(unsigned int) * TM_MAXNB) == cudaSuccess
           && cudaMemset(c->d_scal, 0, TM_MAXNB * sizeof(CgScalars)) == cudaSuccess;
    for (int i = 0; ok && i < TM_NEVENTS; i++) ok = cudaEventCreate(&c->ev[i]) == cudaSuccess;
    if (ok && lane > 0) ok = cudaStreamCreateWithFlags(&c->lane_stream, cudaStreamNonBlocking) == cudaSuccess;
    return ok;
}

static void lane_park(tm_ctx* c, TmLane* L) {          // active fields -> L
    L->ready = 1;
    L->d_partials = c->d_partials; L->d_counter = c->d_counter; L->d_scal = c->d_scal; L->h_scal = c->h_scal;
    memcpy(L->scratch, c->scratch, sizeof(c->scratch));
    memcpy(L->scratch_bytes, c->scratch_bytes, sizeof(c->scratch_bytes));
    memcpy(L->ev, c->ev, sizeof(c->ev));
    L->stream = c->lane_stream;
}
static void lane_load(tm_ctx* c, const TmLane* L) {    // L -> active fields
    c->d_partials = L->d_partials; c->d_counter = L->d_counter; c->d_scal = L->d_scal; c->h_scal = L->h_scal;
    memcpy(c->scratch, L->scratch, sizeof(c->scratch));
    memcpy(c->scratch_bytes, L->scratch_bytes, sizeof(c->scratch_bytes));
    memcpy(c->ev, L->ev, sizeof(c->ev));
    c->lane_stream = L->stream;
}

tm_status tm_lane_use(tm_ctx* c, int lane) {
    if (lane < 0 || lane >= TM_NLANES) return tm_fail(c, TM_EARG, "bad lane");
    if (lane == c->cur_lane) return TM_OK;
    lane_park(c, &c->lanes[c->cur_lane]);
    c->cur_lane = lane;
    if (c->lanes[lane].ready) { lane_load(c, &c->lanes[lane]); return TM_OK; }
    c->d_partials = nullptr; c->d_counter = nullptr; c->d_scal = nullptr; c->h_scal = nullptr;
    memset(c->scratch, 0, sizeof(c->scratch));
    memset(c->scratch_bytes, 0, sizeof(c->scratch_bytes));
    memset(c->ev, 0, sizeof(c->ev));
    c->lane_stream = nullptr;
    if (!lane_alloc(c, lane)) { cudaGetLastError(); return tm_fail(c, TM_EALLOC, "lane: device allocation failed"); }
    return TM_OK;
}

extern "C" tm_status tm_create(tm_ctx** out, const int dims[4], int t_boundary, int device) {
    if (!out || !dims) { snprintf(g_last_error, sizeof(g_last_error), "tm_create: null argument"); return TM_EARG; }
    *out = nullptr;
    for (int i = 0; i < 4; i++)
        if (dims[i] < 2 || (dims[i] & 1)) {
            snprintf(g_last_error, sizeof(g_last_error), "tm_create: extents must be even and >= 2");
            return TM_EDIM;
        }
    if (t_boundary != 1 && t_boundary != -1) {
        snprintf(g_last_error, sizeof(g_last_error), "tm_create: t_boundary must be +1 or -1");
        return TM_EARG;
    }
    const size_t V = (size_t)dims[0] * dims[1] * dims[2] * dims[3];
    // one reduction partial per 128-site Dslash CTA must fit a source's slot of the partials buffer (TM_PSTRIDE)
    if (V / 2 > (size_t)128 * TM_PSTRIDE) { snprintf(g_last_error, sizeof(g_last_error), "tm_create: lattice too large (more than %zu sites)", (size_t)256 * TM_PSTRIDE); return TM_EDIM; }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev <= 0 || device < 0 || device >= ndev) {
        snprintf(g_last_error, sizeof(g_last_error), "tm_create: no usable CUDA device %d (%s); there is no CPU fallback",
                 device, e != cudaSuccess ? cudaGetErrorString(e) : "device count");
        cudaGetLastError();
        return TM_ECUDA;
    }
    e = cudaSetDevice(device);
    if (e != cudaSuccess) { snprintf(g_last_error, sizeof(g_last_error), "cudaSetDevice: %s", cudaGetErrorString(e)); return TM_ECUDA; }
    tm_ctx* c = (tm_ctx*)calloc(1, sizeof(tm_ctx));
    if (!c) return TM_EALLOC;
    for (int i = 0; i < 4; i++) c->X[i] = dims[i];
    c->Xh = dims[0] / 2;
    c->V = V; c->Vh = V / 2;
    c->tb = t_boundary;
    c->device = device;
    cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device);
    bool ok = lane_alloc(c, 0);
    if (!ok) {
        snprintf(g_last_error, sizeof(g_last_error), "tm_create: device allocation failed: %s", cudaGetErrorString(cudaGetLastError()));
        tm_destroy(c);
        return TM_EALLOC;
    }
    *out = c;
    return TM_OK;
}

extern "C" tm_status tm_set_option(tm_ctx* c, tm_option opt, int value) {
    if (!c) return TM_EARG;
    switch (opt) {
        case TM_OPT_GROUP:
            if (value != 0 && value != 1 && value != 2 && value != 4 && value != 8)
                return tm_fail(c, TM_EARG, "tm_set_option: TM_OPT_GROUP must be 0 (automatic), 1, 2, 4 or 8");
            c->opt_group = value;
            return TM_OK;
        case TM_OPT_CONTRACT_PATH:
            if (value < 0 || value > 4) return tm_fail(c, TM_EARG, "tm_set_option: TM_OPT_CONTRACT_PATH must be 0..4");
            c->opt_contract = value;
            return TM_OK;
        case TM_OPT_LANES:
            if (value < 0 || value > TM_NLANES) return tm_fail(c, TM_EARG, "tm_set_option: TM_OPT_LANES must be 0 (automatic), 1 or 2");
            c->opt_lanes = value;
            return TM_OK;
        case TM_OPT_POISON:
            if (value != 0 && value != 1) return tm_fail(c, TM_EARG, "tm_set_option: TM_OPT_POISON must be 0 or 1");
            c->opt_poison = value;
            return TM_OK;
    }
    return tm_fail(c, TM_EARG, "tm_set_option: unknown option");
}

static void drop_gauge_copies(tm_ctx* c) {
    for (int p = 0; p < 4; p++)
        for (int r = 0; r < 2; r++)
            if (c->gauge[p][r]) { cudaFree(c->gauge[p][r]); c->gauge[p][r] = nullptr; c->gauge_valid[p][r] = 0; }
}

extern "C" tm_status tm_destroy(tm_ctx* c) {
    if (!c) return TM_OK;
    cudaSetDevice(c->device);
    cudaDeviceSynchronize();
    drop_gauge_copies(c);
    if (c->d_Ucanon) cudaFree(c->d_Ucanon);
    if (c->master_ev) cudaEventDestroy(c->master_ev);
    for (int p = 0; p < 4; p++)
        for (int r = 0; r < 2; r++)
            if (c->gauge_ev[p][r]) cudaEventDestroy(c->gauge_ev[p][r]);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    lane_park(c, &c->lanes[c->cur_lane]);
    for (int l = 0; l < TM_NLANES; l++) {
        TmLane* L = &c->lanes[l];
        if (!L->ready) continue;
        if (L->d_partials) cudaFree(L->d_partials);
        if (L->d_counter) cudaFree(L->d_counter);
        if (L->d_scal) cudaFree(L->d_scal);
        if (L->h_scal) cudaFreeHost(L->h_scal);
        for (int i = 0; i < TM_MAX_SCRATCH; i++)
            if (L->scratch[i]) cudaFree(L->scratch[i]);
        for (int i = 0; i < TM_NEVENTS; i++)
            if (L->ev[i]) cudaEventDestroy(L->ev[i]);
        if (L->stream) cudaStreamDestroy(L->stream);
    }
    if (c->d_contract_tables) cudaFree(c->d_contract_tables);
    free(c->h_contract_tables);
    cudaGetLastError();
    free(c);
    return TM_OK;
}

tm_status tm_ws(tm_ctx* c, int slot, size_t bytes, void** out) {
    if (slot < 0 || slot >= TM_MAX_SCRATCH) return tm_fail(c, TM_EARG, "bad workspace slot");
    if (c->scratch_bytes[slot] < bytes) {
        if (c->scratch[slot]) {
            cudaDeviceSynchronize();      // a running kernel may still use the old block
            cudaFree(c->scratch[slot]);
            c->scratch[slot] = nullptr; c->scratch_bytes[slot] = 0;
        }
        cudaError_t e = cudaMalloc(&c->scratch[slot], bytes);
        if (e != cudaSuccess) { cudaGetLastError(); c->scratch[slot] = nullptr; return tm_fail(c, TM_EALLOC, "workspace: out of device memory"); }
        c->scratch_bytes[slot] = bytes;
        // TM_OPT_POISON: fresh workspaces start as NaN in every storage precision (0xFF bytes), so a kernel that reads
        // workspace memory nothing has written yet shows up in the results instead of seeing the driver's zero pages
        if (c->opt_poison && cudaMemset(c->scratch[slot], 0xFF, bytes) != cudaSuccess)
            return tm_cuda_fail(c, cudaGetLastError(), "workspace poison");
    }
    *out = c->scratch[slot];
    return TM_OK;
}

// A new master: the reduced-precision copies keep their allocations and are marked stale (repacked from the master on
// their next use, on the stream of that use), so loading a gauge field costs one copy and no synchronisation.
static tm_status load_gauge_impl(tm_ctx* c, const void* U, cudaMemcpyKind kind, cudaStream_t st) {
    TM_CUDA(c, cudaSetDevice(c->device));
    const size_t bytes = c->V * 4 * 9 * 16;
    if (!c->d_Ucanon) {
        cudaError_t e = cudaMalloc(&c->d_Ucanon, bytes);
        if (e != cudaSuccess) { cudaGetLastError(); c->d_Ucanon = nullptr; return tm_fail(c, TM_EALLOC, "tm_load_gauge: out of device memory"); }
    }
    memset(c->gauge_valid, 0, sizeof(c->gauge_valid));
    // packs of the previous master that were enqueued on other streams must have read it before it is overwritten
    for (int p = 0; p < 4; p++)
        for (int r = 0; r < 2; r++)
            if (c->gauge_ev[p][r] && c->gauge_st[p][r] != st) TM_CUDA(c, cudaStreamWaitEvent(st, c->gauge_ev[p][r], 0));
    TM_CUDA(c, cudaMemcpyAsync(c->d_Ucanon, U, bytes, kind, st));
    if (!c->master_ev) TM_CUDA(c, cudaEventCreateWithFlags(&c->master_ev, cudaEventDisableTiming));
    TM_CUDA(c, cudaEventRecord(c->master_ev, st));
    c->master_st = st;
    return TM_OK;
}

extern "C" tm_status tm_load_gauge(tm_ctx* c, const void* d_U, void* stream) {
    if (!c || !d_U) return tm_fail(c, TM_EARG, "tm_load_gauge: null argument");
    return load_gauge_impl(c, d_U, cudaMemcpyDeviceToDevice, (cudaStream_t)stream);
}

extern "C" tm_status tm_load_gauge_host(tm_ctx* c, const void* h_U, void* stream) {
    if (!c || !h_U) return tm_fail(c, TM_EARG, "tm_load_gauge_host: null argument");
    return load_gauge_impl(c, h_U, cudaMemcpyHostToDevice, (cudaStream_t)stream);
}

extern "C" size_t tm_field_bytes(const tm_ctx* c, tm_prec prec, int full_lattice) {
    if (!c || (int)prec < 0 || (int)prec > 3) return 0;
    return tm_parity_bytes(c, prec) * (full_lattice ? 2 : 1);
}

extern "C" tm_status tm_field_import(tm_ctx* c, void* d_internal, const void* d_canon, tm_prec prec, void* stream) {
    if (!c || !d_internal || !d_canon) return tm_fail(c, TM_EARG, "tm_field_import: null argument");
    TM_CUDA(c, cudaSetDevice(c->device));
    return tm_import_launch(c, d_internal, d_canon, prec, (cudaStream_t)stream);
}

extern "C" tm_status tm_field_export(tm_ctx* c, void* d_canon, const void* d_internal, tm_prec prec, void* stream) {
    if (!c || !d_internal || !d_canon) return tm_fail(c, TM_EARG, "tm_field_export: null argument");
    TM_CUDA(c, cudaSetDevice(c->device));
    return tm_export_launch(c, d_canon, d_internal, prec, (cudaStream_t)stream);
}

// Row f3 (multi-source Dslash): the same operator pieces as tm_dslash (HOP, HOP_TWINV, XPAY; reconstruct-12) on nb
// stacked parity fields per launch -- source b's in / x / out sit b parity fields (tm_field_bytes(prec, 0)) behind
// source 0's.  CTAs nb*k .. nb*k + nb-1 work on the same 128 sites of the nb sources, so the later readers of every
// link find it in L2 instead of HBM.  Results are bit-identical to nb tm_dslash calls.
extern "C" tm_status tm_dslash_multi(tm_ctx* c, void* d_out, const void* d_in, const void* d_x, int nb, tm_op op,
                                     int out_parity, int dagger, double kappa, double mu, tm_prec prec, void* stream) {
    if (!c || !d_out || !d_in) return tm_fail(c, TM_EARG, "tm_dslash_multi: null argument");
    if (d_out == d_in) return tm_fail(c, TM_EARG, "tm_dslash_multi: out must not alias in");
    if ((int)prec < 0 || (int)prec > 3) return tm_fail(c, TM_EPREC, "tm_dslash_multi: unknown precision");
    if (nb < 1 || nb > TM_MAXNB || (nb & (nb - 1))) return tm_fail(c, TM_EARG, "tm_dslash_multi: nb must be 1, 2, 4 or 8");
    if (op == TM_OP_XPAY && !d_x) return tm_fail(c, TM_EARG, "tm_dslash_multi: XPAY needs x");
    cudaStream_t st = (cudaStream_t)stream;
    TM_CUDA(c, cudaSetDevice(c->device));
    DslashCall k;
    memset(&k, 0, sizeof(k));
    k.out = d_out; k.in = d_in; k.x = nullptr;
    k.out_parity = out_parity & 1; k.dagger = dagger ? 1 : 0;
    k.kappa = kappa; k.mu = mu; k.coef = 1.0; k.red_op = RED_NONE;
    switch (op) {
        case TM_OP_HOP: break;
        case TM_OP_HOP_TWINV: k.post = 1; break;
        case TM_OP_XPAY: k.x = d_x; k.xmode = 2; k.coef = -kappa * kappa; break;
        default: return tm_fail(c, TM_EARG, "tm_dslash_multi: op must be HOP, HOP_TWINV or XPAY");
    }
    c->nb = nb;
    const tm_status s = tm_dslash_launch(c, k, prec, TM_R12, st);
    c->nb = 1;
    return s;
}

extern "C" tm_status tm_dslash(tm_ctx* c, void* d_out, const void* d_in, const void* d_x, tm_op op,
                               int out_parity, int dagger, double kappa, double mu, tm_prec prec,
                               tm_recon recon, void* stream) {
    if (!c || !d_out || !d_in) return tm_fail(c, TM_EARG, "tm_dslash: null argument");
    if (d_out == d_in) return tm_fail(c, TM_EARG, "tm_dslash: out must not alias in");
    if ((int)prec < 0 || (int)prec > 3) return tm_fail(c, TM_EPREC, "tm_dslash: unknown precision");
    if (recon != TM_R12 && recon != TM_R18) return tm_fail(c, TM_EARG, "tm_dslash: recon must be 12 or 18");
    if (op == TM_OP_XPAY && !d_x) return tm_fail(c, TM_EARG, "tm_dslash: XPAY needs x");
    cudaStream_t st = (cudaStream_t)stream;
    TM_CUDA(c, cudaSetDevice(c->device));
    const size_t pb = tm_parity_bytes(c, prec);
    DslashCall k;
    memset(&k, 0, sizeof(k));
    k.out = d_out; k.in = d_in; k.x = nullptr;
    k.out_parity = out_parity & 1; k.dagger = dagger ? 1 : 0;
    k.kappa = kappa; k.mu = mu; k.coef = 1.0; k.red_op = RED_NONE;
    switch (op) {
        case TM_OP_HOP: return tm_dslash_launch(c, k, prec, recon, st);
        case TM_OP_HOP_TWINV: k.post = 1; return tm_dslash_launch(c, k, prec, recon, st);
        case TM_OP_XPAY: k.x = d_x; k.xmode = 2; k.coef = -kappa * kappa; return tm_dslash_launch(c, k, prec, recon, st);
        case TM_OP_M_FULL: {
            // out_p = A in_p - kappa D_pq in_q for both parities
            for (int p = 0; p < 2; p++) {
                k.out = (char*)d_out + p * pb;
                k.in = (const char*)d_in + (1 - p) * pb;
                k.x = (const char*)d_in + p * pb;
                k.out_parity = p; k.xmode = 2; k.coef = -kappa;
                TM_TRY(tm_dslash_launch(c, k, prec, recon, st));
            }
            return TM_OK;
        }
        case TM_OP_MHAT: {
            void* tmp;
            TM_TRY(tm_ws(c, WS_API_A, pb, &tmp));
            k.out = tmp; k.out_parity = 1; k.post = 1;
            TM_TRY(tm_dslash_launch(c, k, prec, recon, st));
            k.out = d_out; k.in = tmp; k.x = d_in; k.out_parity = 0; k.post = 0; k.xmode = 2; k.coef = -kappa * kappa;
            return tm_dslash_launch(c, k, prec, recon, st);
        }
    }
    return tm_fail(c, TM_EARG, "tm_dslash: unknown op");
}
