// contract.cuh -- device helpers shared by the two contraction kernels (contract.cu: generic path,
// contract_tma.cu: TMA-staged fast path): packed complex-pair arithmetic, SU(3) x spinor, the
// colour-traced outer product and the row-buffer geometry.
#pragma once
#include "kernels.h"
#include "su3.cuh"

#define CT_THREADS 320          // real components per site: 10 (fam, d) x 16 complex x 2
#define CT_NCC 160              // complex components per site
#define CT_NC 5                 // consumer warps: one thread per complex component
#define CT_BSC 34               // row-buffer stride in complex numbers (32 x-values + 2 pad: conflict-free 16-byte reads)

template <int PRUNE> struct QLayout { static constexpr int NQ = PRUNE ? 29 : 49; };

struct ContractArgs {
    const void* s;         // full-lattice internal field (even block, odd block)
    const void* eta;
    const void* gauge;
    void* qbuf;            // [T*Lz][NQ][320]
    const void* wx;        // [Lx][8]: 1, c1, s1, c2, s2, c3, s3, 0   (F precision)
    const void* wy;        // [Ly][8]
    Geom g;
    double tb;
    int t_first;           // first timeslice of the launch (grid = Lz x number of timeslices)
};

// ---- pair arithmetic: one complex number (re, im) per pair.  fp32 pairs live in one 64-bit register
// and use Blackwell's packed FFMA2 / FADD2 (PTX fma.rn.f32x2): one issue slot per complex FMA with a
// broadcast real scalar; ptxas folds the (re, im) swap into the operand swizzle.
template <typename F> struct P2;
template <> struct P2<float> {
    typedef unsigned long long T;
    static __device__ __forceinline__ T make(float re, float im) { T r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(re), "f"(im)); return r; }
    static __device__ __forceinline__ void get(T v, float& re, float& im) { asm("mov.b64 {%0, %1}, %2;" : "=f"(re), "=f"(im) : "l"(v)); }
    static __device__ __forceinline__ T fma_s(float s, T b, T c) {      // c + s * b
        T d; const T ss = make(s, s);
        asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(ss), "l"(b), "l"(c));
        return d;
    }
    static __device__ __forceinline__ T add(T a, T b) { T d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
    static __device__ __forceinline__ T mul_s(float s, T b) { T d; const T ss = make(s, s); asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(ss), "l"(b)); return d; }
    // c + s * (i b) = (c.re - s b.im, c.im + s b.re): two scalar FFMA on the halves of the pairs -- the same fp32-pipe
    // time as one FFMA2, and no (-im, re) pair has to be built first (a negation and a register move per operand)
    static __device__ __forceinline__ T fma_si(float s, T b, T c) {
        float br, bi, cr, ci;
        get(b, br, bi); get(c, cr, ci);
        return make(fmaf(-s, bi, cr), fmaf(s, br, ci));
    }
};
template <> struct P2<double> {
    typedef double2 T;
    static __device__ __forceinline__ T make(double re, double im) { return make_double2(re, im); }
    static __device__ __forceinline__ void get(T v, double& re, double& im) { re = v.x; im = v.y; }
    static __device__ __forceinline__ T fma_s(double s, T b, T c) { return make_double2(fma(s, b.x, c.x), fma(s, b.y, c.y)); }
    static __device__ __forceinline__ T add(T a, T b) { return make_double2(a.x + b.x, a.y + b.y); }
    static __device__ __forceinline__ T mul_s(double s, T b) { return make_double2(s * b.x, s * b.y); }
    static __device__ __forceinline__ T fma_si(double s, T b, T c) { return make_double2(fma(-s, b.y, c.x), fma(s, b.x, c.y)); }
};
// i * v = (-im, re)
template <typename F> __device__ __forceinline__ typename P2<F>::T times_i(typename P2<F>::T v) {
    F re, im;
    P2<F>::get(v, re, im);
    return P2<F>::make(-im, re);
}

// out[sp][a] (+|-)= sum_b U[a][b] in[sp][b]  (DAG: U^dag), 4 spins x 3 colours as 12 pairs; NEG subtracts.
// Loop order: the 12 accumulators are updated round-robin, so consecutive FFMA2 are independent
// (a dependent chain per output would expose the FFMA2 latency: few warps per SM in these kernels).
template <int DAG, int NEG, typename F>
__device__ __forceinline__ void su3_macc(const F* U, const typename P2<F>::T* in, typename P2<F>::T* out) {
    typedef typename P2<F>::T T;
#pragma unroll
    for (int b = 0; b < 3; b++) {
        F ur[3], ui[3];
#pragma unroll
        for (int a = 0; a < 3; a++) {
            ur[a] = DAG ? U[(b * 3 + a) * 2] : U[(a * 3 + b) * 2];
            ui[a] = DAG ? -U[(b * 3 + a) * 2 + 1] : U[(a * 3 + b) * 2 + 1];
            if (NEG) { ur[a] = -ur[a]; ui[a] = -ui[a]; }
        }
        // (ur + i ui) * in = ur * in + ui * (i in)
#pragma unroll
        for (int a = 0; a < 3; a++)
#pragma unroll
            for (int sp = 0; sp < 4; sp++) out[sp * 3 + a] = P2<F>::fma_s(ur[a], in[sp * 3 + b], out[sp * 3 + a]);
#pragma unroll
        for (int a = 0; a < 3; a++)
#pragma unroll
            for (int sp = 0; sp < 4; sp++) out[sp * 3 + a] = P2<F>::fma_si(ui[a], in[sp * 3 + b], out[sp * 3 + a]);
    }
}

template <typename S>
__device__ __forceinline__ void load_spinor_pairs(const S* f, size_t Vh, size_t h, typename P2<S>::T* v) {
    S t[24];
    load_spinor<S>(f, Vh, h, t);
#pragma unroll
    for (int i = 0; i < 12; i++) v[i] = P2<S>::make(t[2 * i], t[2 * i + 1]);
}

__device__ __forceinline__ void named_bar_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
__device__ __forceinline__ void named_bar_arrive(int id, int count) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory"); }

// C[a][b] = sum_c conj(s_ac) psi_bc for the (fam, d) slot `slot` of site column `lane` -> row buffer
// (16 independent accumulators updated round-robin, see su3_macc)
template <typename F>
__device__ __forceinline__ void outer_store(const typename P2<F>::T* sv, const typename P2<F>::T* psi,
                                            typename P2<F>::T* rowbuf, int slot, int lane) {
    typedef typename P2<F>::T T;
    T acc[16];
#pragma unroll
    for (int i = 0; i < 16; i++) acc[i] = P2<F>::make(0, 0);
#pragma unroll
    for (int c = 0; c < 3; c++) {
        F sre[4], sim[4];
#pragma unroll
        for (int a = 0; a < 4; a++) { P2<F>::get(sv[a * 3 + c], sre[a], sim[a]); sim[a] = -sim[a]; }
        // conj(s) psi = s.re * psi - s.im * (i psi)
#pragma unroll
        for (int a = 0; a < 4; a++)
#pragma unroll
            for (int bb = 0; bb < 4; bb++) acc[a * 4 + bb] = P2<F>::fma_s(sre[a], psi[bb * 3 + c], acc[a * 4 + bb]);
#pragma unroll
        for (int a = 0; a < 4; a++)
#pragma unroll
            for (int bb = 0; bb < 4; bb++) acc[a * 4 + bb] = P2<F>::fma_si(sim[a], psi[bb * 3 + c], acc[a * 4 + bb]);
    }
    T* out = rowbuf + (size_t)(slot * 16) * CT_BSC + lane;
#pragma unroll
    for (int i = 0; i < 16; i++) out[(size_t)i * CT_BSC] = acc[i];
}
