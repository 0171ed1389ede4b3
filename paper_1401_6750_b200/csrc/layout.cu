// layout.cu -- canonical <-> internal layout conversion, gauge packing, Z4 noise expansion.
// (SURVEY.md sec 8b "Boundary", "Input recipe".)
#include "kernels.h"

__device__ __forceinline__ int site_coords(const Geom& g, int par, int h, int& lex) {     // returns t
    int q = h / g.Xh;
    const int y = q % g.X1; q /= g.X1;
    const int z = q % g.X2;
    const int t = q / g.X2;
    lex = 2 * h + ((y + z + t + par) & 1);
    return t;
}

template <typename S, int R>
__global__ void gauge_pack_kernel(const double* __restrict__ Uc, S* __restrict__ out, Geom g) {
    typedef typename Prec<S>::F F;
    constexpr int GCV = GaugeLayout<S, R>::GCV;
    constexpr int NCH = GaugeLayout<S, R>::NCH;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 8L * g.Vh) return;
    const int h = (int)(idx % g.Vh);
    const int mu = (int)((idx / g.Vh) & 3);
    const int par = (int)(idx / (4L * g.Vh));
    int lex;
    site_coords(g, par, h, lex);
    const double* src = Uc + ((size_t)lex * 4 + mu) * 18;
    F u[18];
#pragma unroll
    for (int i = 0; i < R; i++) u[i] = (F)src[i];
    S* base = out + ((size_t)(par * 4 + mu) * NCH * g.Vh + h) * GCV;
#pragma unroll
    for (int k = 0; k < NCH; k++) VecIO<S, GCV, LD_DEFAULT>::st(base + (size_t)k * g.Vh * GCV, u + k * GCV);
}

template <typename S, int R>
static tm_status gauge_pack_t(tm_ctx* ctx, void** slot, cudaStream_t st) {
    const size_t bytes = (size_t)8 * ctx->Vh * R * sizeof(S);
    if (!*slot) {
        cudaError_t e = cudaMalloc(slot, bytes);
        if (e != cudaSuccess) { *slot = nullptr; cudaGetLastError(); return tm_fail(ctx, TM_EALLOC, "gauge copy: out of device memory"); }
    }
    const long n = 8L * ctx->Vh;
    gauge_pack_kernel<S, R><<<(unsigned)((n + 255) / 256), 256, 0, st>>>((const double*)ctx->d_Ucanon, (S*)*slot, tm_geom(ctx));
    TM_LAUNCH_CHECK(ctx, "gauge_pack_kernel");
    return TM_OK;
}

tm_status tm_get_gauge(tm_ctx* ctx, tm_prec prec, tm_recon recon, cudaStream_t st, const void** out) {
    if (!ctx->d_Ucanon) return tm_fail(ctx, TM_EARG, "no gauge field loaded (call tm_load_gauge first)");
    if (recon != TM_R12 && recon != TM_R18) return tm_fail(ctx, TM_EARG, "recon must be 12 or 18");
    if ((int)prec < 0 || (int)prec > 3) return tm_fail(ctx, TM_EPREC, "unknown precision");
    const int r = (recon == TM_R12) ? 1 : 0;
    void** slot = &ctx->gauge[prec][r];
    if (!*slot || !ctx->gauge_valid[prec][r]) {
        // the master may have been uploaded on another stream
        if (ctx->master_ev && ctx->master_st != st) TM_CUDA(ctx, cudaStreamWaitEvent(st, ctx->master_ev, 0));
        tm_status s = TM_OK;
        switch (prec) {
            case TM_F64:  s = r ? gauge_pack_t<double, 12>(ctx, slot, st) : gauge_pack_t<double, 18>(ctx, slot, st); break;
            case TM_F32:  s = r ? gauge_pack_t<float, 12>(ctx, slot, st) : gauge_pack_t<float, 18>(ctx, slot, st); break;
            case TM_F16:  s = r ? gauge_pack_t<__half, 12>(ctx, slot, st) : gauge_pack_t<__half, 18>(ctx, slot, st); break;
            case TM_BF16: s = r ? gauge_pack_t<__nv_bfloat16, 12>(ctx, slot, st) : gauge_pack_t<__nv_bfloat16, 18>(ctx, slot, st); break;
        }
        TM_TRY(s);
        ctx->gauge_valid[prec][r] = 1;
        if (!ctx->gauge_ev[prec][r]) TM_CUDA(ctx, cudaEventCreateWithFlags(&ctx->gauge_ev[prec][r], cudaEventDisableTiming));
        TM_CUDA(ctx, cudaEventRecord(ctx->gauge_ev[prec][r], st));
        ctx->gauge_st[prec][r] = st;
    } else if (ctx->gauge_ev[prec][r] && ctx->gauge_st[prec][r] != st) {
        // packed on another stream: order this stream after the pack (a no-op once the pack has finished)
        TM_CUDA(ctx, cudaStreamWaitEvent(st, ctx->gauge_ev[prec][r], 0));
    }
    *out = *slot;
    return TM_OK;
}

// ------------------------------------------------------------------ spinor import / export
template <typename S>
__global__ void import_kernel(const double* __restrict__ canon, S* __restrict__ f, Geom g) {
    typedef typename Prec<S>::F F;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 2L * g.Vh) return;
    const int par = (int)(idx / g.Vh), h = (int)(idx % g.Vh);
    int lex;
    site_coords(g, par, h, lex);
    F v[24];
#pragma unroll
    for (int i = 0; i < 24; i++) v[i] = (F)canon[(size_t)lex * 24 + i];
    store_spinor<S>(f + (size_t)par * g.Vh * 24, g.Vh, h, v);
}

template <typename S>
__global__ void export_kernel(double* __restrict__ canon, const S* __restrict__ f, Geom g) {
    typedef typename Prec<S>::F F;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 2L * g.Vh) return;
    const int par = (int)(idx / g.Vh), h = (int)(idx % g.Vh);
    int lex;
    site_coords(g, par, h, lex);
    F v[24];
    load_spinor<S>(f + (size_t)par * g.Vh * 24, g.Vh, h, v);
#pragma unroll
    for (int i = 0; i < 24; i++) canon[(size_t)lex * 24 + i] = (double)v[i];
}

tm_status tm_import_launch(tm_ctx* ctx, void* d_int, const void* d_canon, tm_prec prec, cudaStream_t st) {
    const long n = 2L * ctx->Vh;
    const unsigned grid = (unsigned)((n + 127) / 128);
    const Geom g = tm_geom(ctx);
    switch (prec) {
        case TM_F64:  import_kernel<double><<<grid, 128, 0, st>>>((const double*)d_canon, (double*)d_int, g); break;
        case TM_F32:  import_kernel<float><<<grid, 128, 0, st>>>((const double*)d_canon, (float*)d_int, g); break;
        case TM_F16:  import_kernel<__half><<<grid, 128, 0, st>>>((const double*)d_canon, (__half*)d_int, g); break;
        case TM_BF16: import_kernel<__nv_bfloat16><<<grid, 128, 0, st>>>((const double*)d_canon, (__nv_bfloat16*)d_int, g); break;
        default: return tm_fail(ctx, TM_EPREC, "tm_field_import: unknown precision");
    }
    TM_LAUNCH_CHECK(ctx, "import_kernel");
    return TM_OK;
}

tm_status tm_export_launch(tm_ctx* ctx, void* d_canon, const void* d_int, tm_prec prec, cudaStream_t st) {
    const long n = 2L * ctx->Vh;
    const unsigned grid = (unsigned)((n + 127) / 128);
    const Geom g = tm_geom(ctx);
    switch (prec) {
        case TM_F64:  export_kernel<double><<<grid, 128, 0, st>>>((double*)d_canon, (const double*)d_int, g); break;
        case TM_F32:  export_kernel<float><<<grid, 128, 0, st>>>((double*)d_canon, (const float*)d_int, g); break;
        case TM_F16:  export_kernel<__half><<<grid, 128, 0, st>>>((double*)d_canon, (const __half*)d_int, g); break;
        case TM_BF16: export_kernel<__nv_bfloat16><<<grid, 128, 0, st>>>((double*)d_canon, (const __nv_bfloat16*)d_int, g); break;
        default: return tm_fail(ctx, TM_EPREC, "tm_field_export: unknown precision");
    }
    TM_LAUNCH_CHECK(ctx, "export_kernel");
    return TM_OK;
}

// ------------------------------------------------------------------ Z4 noise
// mix = splitmix64 finaliser, h(seed, r, c) = mix(mix(seed*G + r) + c),
// eta[c] = i^(h & 3), c = (lex*4 + spin)*3 + col.  `base` = mix(seed*G + r) is computed on the host.
__host__ __device__ __forceinline__ unsigned long long mix64(unsigned long long z) {
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27; z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}

// t_only >= 0: time dilution -- the noise restricted to timeslice t_only, zero elsewhere
template <typename S>
__global__ void z4_expand_kernel(S* __restrict__ f, const unsigned char* __restrict__ packed,
                                 unsigned long long base, Geom g, int t_only) {
    typedef typename Prec<S>::F F;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 2L * g.Vh) return;
    const int par = (int)(idx / g.Vh), h = (int)(idx % g.Vh);
    int lex;
    const int t = site_coords(g, par, h, lex);
    if (t_only >= 0 && t != t_only) {
        F v[24];
#pragma unroll
        for (int i = 0; i < 24; i++) v[i] = F(0);
        store_spinor<S>(f + (size_t)par * g.Vh * 24, g.Vh, h, v);
        return;
    }
    unsigned int bits = 0;     // 12 exponents, 2 bits each
    if (packed) {
        const unsigned char* p = packed + (size_t)lex * 3;
        bits = (unsigned)p[0] | ((unsigned)p[1] << 8) | ((unsigned)p[2] << 16);
    } else {
#pragma unroll
        for (int c = 0; c < 12; c++)
            bits |= (unsigned)(mix64(base + (unsigned long long)lex * 12ULL + c) & 3ULL) << (2 * c);
    }
    F v[24];
#pragma unroll
    for (int c = 0; c < 12; c++) {
        const unsigned k = (bits >> (2 * c)) & 3u;
        v[2 * c] = (k == 0) ? F(1) : (k == 2) ? F(-1) : F(0);
        v[2 * c + 1] = (k == 1) ? F(1) : (k == 3) ? F(-1) : F(0);
    }
    store_spinor<S>(f + (size_t)par * g.Vh * 24, g.Vh, h, v);
}

tm_status tm_z4_expand(tm_ctx* ctx, void* d_int, tm_prec prec, const unsigned char* d_z4,
                       unsigned long long seed, unsigned long long r, cudaStream_t st, int t_only) {
    const unsigned long long base = mix64(seed * 0x9E3779B97F4A7C15ULL + r);
    const long n = 2L * ctx->Vh;
    const unsigned grid = (unsigned)((n + 127) / 128);
    const Geom g = tm_geom(ctx);
    switch (prec) {
        case TM_F64: z4_expand_kernel<double><<<grid, 128, 0, st>>>((double*)d_int, d_z4, base, g, t_only); break;
        case TM_F32: z4_expand_kernel<float><<<grid, 128, 0, st>>>((float*)d_int, d_z4, base, g, t_only); break;
        default: return tm_fail(ctx, TM_EPREC, "z4 expand: precision must be f32 or f64");
    }
    TM_LAUNCH_CHECK(ctx, "z4_expand_kernel");
    return TM_OK;
}
