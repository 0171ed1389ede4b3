// common.cuh -- context, layouts and vector load/store helpers of libtmloops (sm_100a).
//
// Internal layouts:
//   parity spinor  [24/CV chunks][Vh sites] x (CV reals = 16 bytes), real index r = (spin*3+col)*2 + reim,
//                  chunk k holds reals [k*CV, (k+1)*CV)
//   gauge          [2 parity][4 mu][R/GCV chunks][Vh] x (GCV reals), real index r = (row*3+col)*2 + reim,
//                  R = 12 (rows 0,1) or 18; link U_mu(x) is stored at the parity/half-index of x
//   half index     h = lex/2, lex = ((t*Lz+z)*Ly+y)*Lx+x,  x = 2*(h % Xh) + ((y+z+t+parity)&1)
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include "../../include/tmloops.h"

#define TM_MAX_SCRATCH 48

struct CgScalars;   // blas.cuh

// Launch plan of the CG: the iteration counts at which the previous solve with the same parameters
// paused for a reliable update.  The next solve enqueues its kernels along this plan without
// waiting for the device (every kernel is guarded by the device-side state, so a wrong plan costs
// only no-op launches or an extra host round trip, never a different result).
#define CG_MAX_PAUSES 48
#define TM_NPLANS 6
struct CgPlan {
    int valid;
    int sloppy, outer, recon, max_iter;
    double rho, delta;
    int n_pause;
    int pause_iter[CG_MAX_PAUSES];
};

// A lane = everything one in-flight solve + contraction needs privately: reduction scratch, the device state
// of the CG, workspaces, events and (lanes >= 1) a stream.  The context's own fields of the same names are
// the ACTIVE lane's (tm_lane_use swaps them), so kernels and helpers never see lanes; tsm.cu keeps
// TM_NLANES sources in flight so that the tail of one kernel overlaps the next kernel of another source.
#define TM_NLANES 2
#define TM_NEVENTS 6
struct TmLane {
    int ready;
    double* d_partials;
    unsigned int* d_counter;
    CgScalars* d_scal;
    CgScalars* h_scal;
    void* scratch[TM_MAX_SCRATCH];
    size_t scratch_bytes[TM_MAX_SCRATCH];
    cudaEvent_t ev[TM_NEVENTS];
    cudaStream_t stream;            // owned side stream (lane 0: none, it runs on the caller's stream)
};

struct tm_ctx {
    int X[4];
    int Xh;
    int tb;
    int device;
    int sm_count;
    size_t V, Vh;
    char err[512];
    long launches;
    void* d_Ucanon;                 // fp64 master, canonical [V][4][3][3] complex128
    void* gauge[4][2];              // [prec][recon==12] internal copies, built lazily
    int gauge_valid[4][2];          // 0: allocated but stale (a new master was loaded) -> repacked on next use
    // cross-stream ordering of the lazily built gauge state: the event recorded after the master upload / after each
    // pack, and the stream it was recorded on; a call on another stream waits on the event before it touches the data
    cudaEvent_t master_ev, gauge_ev[4][2];
    cudaStream_t master_st, gauge_st[4][2];
    cudaStream_t copy_stream;       // host -> device prefetch of the packed noise (tsm_estimate_host), created on first use
    // reduction scratch
    double* d_partials;             // per-block partial sums
    unsigned int* d_counter;        // last-block-done counter
    CgScalars* d_scal;              // device scalars of the running solve
    CgScalars* h_scal;              // pinned mirror
    CgPlan plan[TM_NPLANS];         // launch plans keyed by the full parameter tuple (LP and HP keep their own), round-robin eviction
    int plan_next;
    // generic workspace pool (freed in tm_destroy): named slots grown on demand
    void* scratch[TM_MAX_SCRATCH];
    size_t scratch_bytes[TM_MAX_SCRATCH];
    // contraction tables
    void* d_contract_tables;
    void* h_contract_tables;        // host mirror (rebuild only when the momentum list changes)
    size_t contract_tables_bytes;
    cudaEvent_t ev[TM_NEVENTS];     // 0,1: solve; 2,3: tsm; 4: solver state download; 5: lane join
    int cur_lane;
    int nb;                         // sources per launch of the running solve (0 | 1: one; 2: a pair, see blas.cu)
    TmLane lanes[TM_NLANES];        // parked state of the inactive lanes (the active one lives in the fields above)
    cudaStream_t lane_stream;       // stream owned by the active lane (0 for lane 0)
    int opt_group;                  // TM_OPT_GROUP: 0 = automatic | 1 | 2 | 4 | 8 sources per solve
    int opt_lanes;                  // TM_OPT_LANES: 0 = automatic | 1 | 2 jobs in flight
    int opt_poison;                 // TM_OPT_POISON: fill newly allocated workspaces with 0xFF bytes (NaN)
    int opt_contract;               // TM_OPT_CONTRACT_PATH: 0 = automatic | 1 generic | 2 TMA + fp32-pipe DFT | 3 TMA + tensor-core DFT (contract_mma.cu)
};

static inline tm_status tm_fail(tm_ctx* c, tm_status s, const char* msg) {
    if (c) snprintf(c->err, sizeof(c->err), "%s", msg);
    return s;
}
static inline tm_status tm_cuda_fail(tm_ctx* c, cudaError_t e, const char* where) {
    if (c) snprintf(c->err, sizeof(c->err), "CUDA error at %s: %s", where, cudaGetErrorString(e));
    return TM_ECUDA;
}
#define TM_CUDA(ctx, call)                                                        \
    do {                                                                          \
        cudaError_t e__ = (call);                                                 \
        if (e__ != cudaSuccess) return tm_cuda_fail(ctx, e__, #call);             \
    } while (0)
#define TM_TRY(call)                                                              \
    do {                                                                          \
        tm_status s__ = (call);                                                   \
        if (s__ != TM_OK) return s__;                                             \
    } while (0)
#define TM_LAUNCH_CHECK(ctx, name)                                                \
    do {                                                                          \
        (ctx)->launches++;                                                        \
        cudaError_t e__ = cudaGetLastError();                                     \
        if (e__ != cudaSuccess) return tm_cuda_fail(ctx, e__, name);              \
    } while (0)

// workspace slot ids
enum {
    WS_SL_P = 0, WS_SL_W, WS_SL_Z, WS_SL_TMP, WS_SL_R,         // sloppy parity vectors
    WS_AC_X, WS_AC_R,                                           // accumulate-precision x, r
    WS_OU_Y, WS_OU_B, WS_OU_R, WS_OU_TMP, WS_OU_TMP2,           // outer precision parity vectors
    WS_OU_ETA, WS_OU_S,                                         // outer precision full-lattice fields
    WS_CT_S, WS_CT_ETA, WS_CT_PLANES, WS_CT_OUT,                // contraction
    WS_TSM_ACC, WS_TSM_ETA32, WS_TSM_ETA64, WS_TSM_S32, WS_TSM_S64, WS_TSM_Z4, WS_TSM_KEEP,
    WS_API_A, WS_API_B, WS_API_C,
    WS_TD_ACC, WS_TD_PRIM,                                      // time dilution (dilution.cu), HPE (hpe.cu)
    WS_HPE_A, WS_HPE_B, WS_HPE_C, WS_HPE_TAB                   // HPE: hopping-term ping-pong vectors, tables
};
tm_status tm_ws(tm_ctx* c, int slot, size_t bytes, void** out);     // api.cu
tm_status tm_lane_use(tm_ctx* c, int lane);                          // api.cu: make `lane` the active one
tm_status tm_get_gauge(tm_ctx* c, tm_prec prec, tm_recon recon, cudaStream_t st, const void** out);  // layout.cu

static inline size_t tm_prec_size(tm_prec p) { return p == TM_F64 ? 8 : p == TM_F32 ? 4 : 2; }
static inline size_t tm_parity_bytes(const tm_ctx* c, tm_prec p) { return c->Vh * 24 * tm_prec_size(p); }

// ------------------------------------------------------------------ precision traits
template <typename S> struct Prec;
template <> struct Prec<double>        { typedef double F; static constexpr int CV = 2; };
template <> struct Prec<float>         { typedef float  F; static constexpr int CV = 4; };
template <> struct Prec<__half>        { typedef float  F; static constexpr int CV = 8; };
template <> struct Prec<__nv_bfloat16> { typedef float  F; static constexpr int CV = 8; };

// gauge chunk width in reals: 16-byte chunks when the link size allows, else the largest divisor
template <typename S, int R> struct GaugeLayout {
    static constexpr int GCV = (sizeof(S) == 8) ? 2
                             : (sizeof(S) == 4) ? (R == 12 ? 4 : 2)
                             :                    (R == 12 ? 4 : 2);
    static constexpr int NCH = R / GCV;
};

enum { LD_DEFAULT = 0, LD_STREAM = 1 };

// raw N-byte loads
template <int BYTES, int POLICY> struct RawLoad;
template <int POLICY> struct RawLoad<16, POLICY> {
    typedef uint4 T;
    static __device__ __forceinline__ uint4 ld(const void* p) {
        return POLICY == LD_STREAM ? __ldcs((const uint4*)p) : __ldg((const uint4*)p);
    }
};
template <int POLICY> struct RawLoad<8, POLICY> {
    typedef uint2 T;
    static __device__ __forceinline__ uint2 ld(const void* p) {
        return POLICY == LD_STREAM ? __ldcs((const uint2*)p) : __ldg((const uint2*)p);
    }
};
template <int POLICY> struct RawLoad<4, POLICY> {
    typedef unsigned int T;
    static __device__ __forceinline__ unsigned int ld(const void* p) {
        return POLICY == LD_STREAM ? __ldcs((const unsigned int*)p) : __ldg((const unsigned int*)p);
    }
};

__device__ __forceinline__ void cvt_pair(unsigned int w, const __half*, float& a, float& b) {
    float2 f = __half22float2(*reinterpret_cast<__half2*>(&w));
    a = f.x; b = f.y;
}
__device__ __forceinline__ void cvt_pair(unsigned int w, const __nv_bfloat16*, float& a, float& b) {
    // bf16 -> fp32 is a 16-bit shift
    a = __uint_as_float(w << 16);
    b = __uint_as_float(w & 0xffff0000u);
}
__device__ __forceinline__ unsigned int pack_pair(float a, float b, const __half*) {
    __half2 h = __floats2half2_rn(a, b);
    return *reinterpret_cast<unsigned int*>(&h);
}
__device__ __forceinline__ unsigned int pack_pair(float a, float b, const __nv_bfloat16*) {
    __nv_bfloat162 h = __floats2bfloat162_rn(a, b);
    return *reinterpret_cast<unsigned int*>(&h);
}

// load N reals of storage type S (N*sizeof(S) in {4,8,16}) from an aligned address into F out[N]
template <typename S, int N, int POLICY> struct VecIO;

template <int N, int POLICY> struct VecIO<double, N, POLICY> {   // N == 2
    static __device__ __forceinline__ void ld(const double* p, double* out) {
        uint4 v = RawLoad<16, POLICY>::ld(p);
        out[0] = __hiloint2double(v.y, v.x);
        out[1] = __hiloint2double(v.w, v.z);
    }
    static __device__ __forceinline__ void st(double* p, const double* in) {
        *reinterpret_cast<double2*>(p) = make_double2(in[0], in[1]);
    }
};
template <int POLICY> struct VecIO<float, 4, POLICY> {
    static __device__ __forceinline__ void ld(const float* p, float* out) {
        uint4 v = RawLoad<16, POLICY>::ld(p);
        out[0] = __uint_as_float(v.x); out[1] = __uint_as_float(v.y);
        out[2] = __uint_as_float(v.z); out[3] = __uint_as_float(v.w);
    }
    static __device__ __forceinline__ void st(float* p, const float* in) {
        *reinterpret_cast<float4*>(p) = make_float4(in[0], in[1], in[2], in[3]);
    }
};
template <int POLICY> struct VecIO<float, 2, POLICY> {
    static __device__ __forceinline__ void ld(const float* p, float* out) {
        uint2 v = RawLoad<8, POLICY>::ld(p);
        out[0] = __uint_as_float(v.x); out[1] = __uint_as_float(v.y);
    }
    static __device__ __forceinline__ void st(float* p, const float* in) {
        *reinterpret_cast<float2*>(p) = make_float2(in[0], in[1]);
    }
};
template <typename S, int POLICY> struct VecIO<S, 8, POLICY> {   // 16-bit, 16 bytes
    static __device__ __forceinline__ void ld(const S* p, float* out) {
        uint4 v = RawLoad<16, POLICY>::ld(p);
        cvt_pair(v.x, (const S*)0, out[0], out[1]); cvt_pair(v.y, (const S*)0, out[2], out[3]);
        cvt_pair(v.z, (const S*)0, out[4], out[5]); cvt_pair(v.w, (const S*)0, out[6], out[7]);
    }
    static __device__ __forceinline__ void st(S* p, const float* in) {
        uint4 v;
        v.x = pack_pair(in[0], in[1], (const S*)0); v.y = pack_pair(in[2], in[3], (const S*)0);
        v.z = pack_pair(in[4], in[5], (const S*)0); v.w = pack_pair(in[6], in[7], (const S*)0);
        *reinterpret_cast<uint4*>(p) = v;
    }
};
template <int POLICY> struct VecIO<__half, 4, POLICY> {
    static __device__ __forceinline__ void ld(const __half* p, float* out) {
        uint2 v = RawLoad<8, POLICY>::ld(p);
        cvt_pair(v.x, (const __half*)0, out[0], out[1]); cvt_pair(v.y, (const __half*)0, out[2], out[3]);
    }
    static __device__ __forceinline__ void st(__half* p, const float* in) {
        uint2 v;
        v.x = pack_pair(in[0], in[1], (const __half*)0); v.y = pack_pair(in[2], in[3], (const __half*)0);
        *reinterpret_cast<uint2*>(p) = v;
    }
};
template <int POLICY> struct VecIO<__nv_bfloat16, 4, POLICY> {
    static __device__ __forceinline__ void ld(const __nv_bfloat16* p, float* out) {
        uint2 v = RawLoad<8, POLICY>::ld(p);
        cvt_pair(v.x, (const __nv_bfloat16*)0, out[0], out[1]);
        cvt_pair(v.y, (const __nv_bfloat16*)0, out[2], out[3]);
    }
    static __device__ __forceinline__ void st(__nv_bfloat16* p, const float* in) {
        uint2 v;
        v.x = pack_pair(in[0], in[1], (const __nv_bfloat16*)0);
        v.y = pack_pair(in[2], in[3], (const __nv_bfloat16*)0);
        *reinterpret_cast<uint2*>(p) = v;
    }
};
template <int POLICY> struct VecIO<__half, 2, POLICY> {
    static __device__ __forceinline__ void ld(const __half* p, float* out) {
        unsigned int v = RawLoad<4, POLICY>::ld(p);
        cvt_pair(v, (const __half*)0, out[0], out[1]);
    }
    static __device__ __forceinline__ void st(__half* p, const float* in) {
        *reinterpret_cast<unsigned int*>(p) = pack_pair(in[0], in[1], (const __half*)0);
    }
};
template <int POLICY> struct VecIO<__nv_bfloat16, 2, POLICY> {
    static __device__ __forceinline__ void ld(const __nv_bfloat16* p, float* out) {
        unsigned int v = RawLoad<4, POLICY>::ld(p);
        cvt_pair(v, (const __nv_bfloat16*)0, out[0], out[1]);
    }
    static __device__ __forceinline__ void st(__nv_bfloat16* p, const float* in) {
        *reinterpret_cast<unsigned int*>(p) = pack_pair(in[0], in[1], (const __nv_bfloat16*)0);
    }
};

// ------------------------------------------------------------------ spinor / link access
// all 24 reals of one site of a parity field
template <typename S, int POLICY = LD_DEFAULT>
__device__ __forceinline__ void load_spinor(const S* f, size_t Vh, size_t h, typename Prec<S>::F* v) {
    constexpr int CV = Prec<S>::CV;
#pragma unroll
    for (int k = 0; k < 24 / CV; k++) VecIO<S, CV, POLICY>::ld(f + ((size_t)k * Vh + h) * CV, v + k * CV);
}
template <typename S>
__device__ __forceinline__ void store_spinor(S* f, size_t Vh, size_t h, const typename Prec<S>::F* v) {
    constexpr int CV = Prec<S>::CV;
#pragma unroll
    for (int k = 0; k < 24 / CV; k++) VecIO<S, CV, LD_DEFAULT>::st(f + ((size_t)k * Vh + h) * CV, v + k * CV);
}
// reals [8g, 8g+8) of one site: the unit of the precision-agnostic BLAS kernels
template <typename S>
__device__ __forceinline__ void load8(const S* f, size_t Vh, size_t h, int g, typename Prec<S>::F* v) {
    constexpr int CV = Prec<S>::CV;
#pragma unroll
    for (int k = 0; k < 8 / CV; k++)
        VecIO<S, CV, LD_DEFAULT>::ld(f + ((size_t)(g * (8 / CV) + k) * Vh + h) * CV, v + k * CV);
}
template <typename S>
__device__ __forceinline__ void store8(S* f, size_t Vh, size_t h, int g, const typename Prec<S>::F* v) {
    constexpr int CV = Prec<S>::CV;
#pragma unroll
    for (int k = 0; k < 8 / CV; k++)
        VecIO<S, CV, LD_DEFAULT>::st(f + ((size_t)(g * (8 / CV) + k) * Vh + h) * CV, v + k * CV);
}

// link (parity par, direction mu, half index h): R stored reals -> 18 reals (row 2 rebuilt for R = 12)
template <typename S, int R, int POLICY = LD_STREAM>
__device__ __forceinline__ void load_link(const S* g, size_t Vh, int par, int mu, size_t h,
                                          typename Prec<S>::F* u) {
    typedef typename Prec<S>::F F;
    constexpr int GCV = GaugeLayout<S, R>::GCV;
    constexpr int NCH = GaugeLayout<S, R>::NCH;
    const S* base = g + ((size_t)(par * 4 + mu) * NCH * Vh + h) * GCV;
#pragma unroll
    for (int k = 0; k < NCH; k++) VecIO<S, GCV, POLICY>::ld(base + (size_t)k * Vh * GCV, u + k * GCV);
    if (R == 12) {
        // row2 = conj(row0 x row1)
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const int i = (c + 1) % 3, j = (c + 2) % 3;
            F ar = u[2 * i], ai = u[2 * i + 1], br = u[6 + 2 * j], bi = u[6 + 2 * j + 1];
            F cr = u[2 * j], ci = u[2 * j + 1], dr = u[6 + 2 * i], di = u[6 + 2 * i + 1];
            // a_i b_j - a_j b_i, one FMA per statement
            F re = ar * br; re -= ai * bi; re -= cr * dr; re += ci * di;
            F im = ar * bi; im += ai * br; im -= cr * di; im -= ci * dr;
            u[12 + 2 * c] = re;
            u[12 + 2 * c + 1] = -im;
        }
    }
}

// site geometry of a parity field
struct Geom {
    int X0, X1, X2, X3;    // Lx, Ly, Lz, T
    int Xh;                // Lx/2
    int Vh;
    int s1, s2, s3;        // half-index strides of y, z, t:  Xh, Xh*Ly, Xh*Ly*Lz
    int sh0, sh1, sh2;     // log2 of Xh, Ly, Lz when all three are powers of two, else sh0 = -1
    unsigned dm[3];        // otherwise: division by the invariant integers Xh, Ly, Lz as multiply-high + add + shift
    int dl[3];             //   q = (umulhi(dm, n) + n) >> dl,  dl = ceil(log2 d),  dm = floor(2^32 (2^dl - d) / d) + 1
};
// n / d for 0 <= n < 2^31 (Granlund-Montgomery: exact for every 32-bit n in its round-up form; t <= n keeps t + n in 32 bits)
__host__ __device__ __forceinline__ int fast_div(int n, unsigned m, int l) {
#ifdef __CUDA_ARCH__
    return (int)((__umulhi(m, (unsigned)n) + (unsigned)n) >> l);
#else
    return (int)(((unsigned)(((unsigned long long)m * (unsigned)n) >> 32) + (unsigned)n) >> l);
#endif
}
// half index -> (xh, y, z, t): shifts and masks where the extents are powers of two, else three divisions by invariant
// integers (a run-time integer division is ~25 instructions: three of them were 5 % of a Dslash kernel)
__host__ __device__ __forceinline__ void site_coords(const Geom& g, int h, int& xh, int& y, int& z, int& t) {
    if (g.sh0 >= 0) {
        xh = h & (g.Xh - 1);
        int q = h >> g.sh0;
        y = q & (g.X1 - 1); q >>= g.sh1;
        z = q & (g.X2 - 1);
        t = q >> g.sh2;
    } else {
        int q = fast_div(h, g.dm[0], g.dl[0]);
        xh = h - q * g.Xh;
        int q1 = fast_div(q, g.dm[1], g.dl[1]);
        y = q - q1 * g.X1;
        t = fast_div(q1, g.dm[2], g.dl[2]);
        z = q1 - t * g.X2;
    }
}
static inline Geom tm_geom(const tm_ctx* c) {
    Geom g;
    g.X0 = c->X[0]; g.X1 = c->X[1]; g.X2 = c->X[2]; g.X3 = c->X[3];
    g.Xh = c->Xh; g.Vh = (int)c->Vh;
    g.s1 = g.Xh; g.s2 = g.Xh * g.X1; g.s3 = g.Xh * g.X1 * g.X2;
    auto lg = [](int v) { int l = 0; while ((1 << l) < v) l++; return (1 << l) == v ? l : -1; };
    g.sh0 = lg(g.Xh); g.sh1 = lg(g.X1); g.sh2 = lg(g.X2);
    if (g.sh0 < 0 || g.sh1 < 0 || g.sh2 < 0) g.sh0 = g.sh1 = g.sh2 = -1;
    const int dv[3] = {g.Xh, g.X1, g.X2};
    for (int i = 0; i < 3; i++) {
        int l = 0;
        while ((1u << l) < (unsigned)dv[i]) l++;
        g.dl[i] = l;
        g.dm[i] = (unsigned)((((unsigned long long)1 << 32) * (((unsigned long long)1 << l) - (unsigned)dv[i])) / (unsigned)dv[i]) + 1u;
    }
    return g;
}
