// dslash.cu -- twisted-mass parity Dslash stencil for sm_100a.
//
// [B:ns]:  M = (1 + 2 i kappa mu g5) - kappa sum_mu [(1-g_mu) U_mu(x) d_{x+mu,y} + (1+g_mu) U_mu^dag(x-mu) d_{x-mu,y}]
// One thread per output site of one parity.  For each of the 8 neighbours the spinor is projected
// to a 2-spin half-spinor with (1 -+ g_mu) (the rank-2 "gamma-projection spin trick"), multiplied
// by the SU(3) link (rebuilt from two rows for reconstruct-12) and reconstructed into the
// accumulator.  HBM-bound: no tensor cores, 16-byte coalesced chunk loads, streaming (evict-first)
// policy for links (zero reuse), default policy for spinors (8-fold reuse served by L1/L2).
//
// Epilogue (runtime-uniform):  res = c * (D in);  xmode 1: res += x;  xmode 2: res += A x;
//                              post 1: res = A^-1 res;  optional ||res||^2 -> per-block partials + reduce_finish_kernel.
// A = 1 + i a g5,  a = 2 kappa mu (sign flipped for dagger),  A^-1 = (1 - i a g5) / (1 + a^2).
//
// Chiral basis (reading 2): g_mu = [[0, B],[B^dag, 0]] with
//   B_x = -i sigma_x, B_y = -i sigma_y, B_z = -i sigma_z, B_t = 1;
//   (1 + s g_mu) psi = (u, s B^dag u),  u = psi_up + s B psi_low.
#include "kernels.h"
#include "su3.cuh"
#include "contract.cuh"      // P2<float>: packed complex-pair arithmetic (FFMA2 / FADD2)

template <typename F> struct DslashArgs {
    const void* in;
    const void* x;
    void* out;
    const void* gauge;
    Geom g;
    int parity;        // parity of the output sites
    F dsign;           // +1, or -1 for dagger
    F tb;              // time boundary sign
    F a;               // twist 2 kappa mu (already multiplied by dsign)
    F c;               // coefficient of D in
    int xmode, post, red_op;
    double* partials;
    unsigned int* counter;
    CgScalars* sc;
    int guard;         // GUARD_* (blas.cuh): skip unless the running solve is in the matching state
    int nb;            // sources per launch (1 | 2): CTAs 2k and 2k+1 work on the same sites of source 0 and 1,
                       // so that the second reader of every link finds it in L2
    size_t fstride;    // bytes of one parity vector; source 1's operands sit mul_* vectors behind source 0's
    int mul_in, mul_x, mul_out;
    int ns;            // dslash16_group_kernel: sources handled one after the other by a CTA (divides nb)
};

// u (2 spins x 3 colours complex = 12 reals) = psi_up + s * B_mu psi_low
template <int MU, typename F>
__device__ __forceinline__ void project(const F* p, F s, F* u) {
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const F p0r = p[2 * c], p0i = p[2 * c + 1], p1r = p[6 + 2 * c], p1i = p[6 + 2 * c + 1];
        const F p2r = p[12 + 2 * c], p2i = p[12 + 2 * c + 1], p3r = p[18 + 2 * c], p3i = p[18 + 2 * c + 1];
        if (MU == 0) {          // B psi_low = (-i psi3, -i psi2)
            u[2 * c] = p0r + s * p3i;      u[2 * c + 1] = p0i - s * p3r;
            u[6 + 2 * c] = p1r + s * p2i;  u[6 + 2 * c + 1] = p1i - s * p2r;
        } else if (MU == 1) {   // (-psi3, psi2)
            u[2 * c] = p0r - s * p3r;      u[2 * c + 1] = p0i - s * p3i;
            u[6 + 2 * c] = p1r + s * p2r;  u[6 + 2 * c + 1] = p1i + s * p2i;
        } else if (MU == 2) {   // (-i psi2, i psi3)
            u[2 * c] = p0r + s * p2i;      u[2 * c + 1] = p0i - s * p2r;
            u[6 + 2 * c] = p1r - s * p3i;  u[6 + 2 * c + 1] = p1i + s * p3r;
        } else {                // (psi2, psi3)
            u[2 * c] = p0r + s * p2r;      u[2 * c + 1] = p0i + s * p2i;
            u[6 + 2 * c] = p1r + s * p3r;  u[6 + 2 * c + 1] = p1i + s * p3i;
        }
    }
}

// acc_up += v ; acc_low += s * B_mu^dag v
template <int MU, typename F>
__device__ __forceinline__ void reconstruct(const F* v, F s, F* acc) {
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const F v0r = v[2 * c], v0i = v[2 * c + 1], v1r = v[6 + 2 * c], v1i = v[6 + 2 * c + 1];
        acc[2 * c] += v0r;      acc[2 * c + 1] += v0i;
        acc[6 + 2 * c] += v1r;  acc[6 + 2 * c + 1] += v1i;
        if (MU == 0) {          // B^dag v = (i v1, i v0)
            acc[12 + 2 * c] -= s * v1i;  acc[12 + 2 * c + 1] += s * v1r;
            acc[18 + 2 * c] -= s * v0i;  acc[18 + 2 * c + 1] += s * v0r;
        } else if (MU == 1) {   // (v1, -v0)
            acc[12 + 2 * c] += s * v1r;  acc[12 + 2 * c + 1] += s * v1i;
            acc[18 + 2 * c] -= s * v0r;  acc[18 + 2 * c + 1] -= s * v0i;
        } else if (MU == 2) {   // (i v0, -i v1)
            acc[12 + 2 * c] -= s * v0i;  acc[12 + 2 * c + 1] += s * v0r;
            acc[18 + 2 * c] += s * v1i;  acc[18 + 2 * c + 1] -= s * v1r;
        } else {                // (v0, v1)
            acc[12 + 2 * c] += s * v0r;  acc[12 + 2 * c + 1] += s * v0i;
            acc[18 + 2 * c] += s * v1r;  acc[18 + 2 * c + 1] += s * v1i;
        }
    }
}

template <int MU, int FWD, typename S, int R>
__device__ __forceinline__ void hop(const S* in, const S* gauge, const Geom& g, int par_out, size_t h_out,
                                    size_t h_nb, typename Prec<S>::F sgn, typename Prec<S>::F bsign,
                                    bool wrap, typename Prec<S>::F* acc) {
    typedef typename Prec<S>::F F;
    F psi[24], u[12], v[12], U[18];
    load_spinor<S>(in, g.Vh, h_nb, psi);
    if (FWD) load_link<S, R>(gauge, g.Vh, par_out, MU, h_out, U);
    else     load_link<S, R>(gauge, g.Vh, 1 - par_out, MU, h_nb, U);
    project<MU>(psi, sgn, u);
    if (MU == 3 && wrap) {
#pragma unroll
        for (int i = 0; i < 12; i++) u[i] *= bsign;
    }
    su3_mul_half<FWD ? 0 : 1>(U, u, v);
    reconstruct<MU>(v, sgn, acc);
}

template <typename S, int R>
__global__ void __launch_bounds__(128) dslash_kernel(DslashArgs<typename Prec<S>::F> A) {
    typedef typename Prec<S>::F F;
    __shared__ double sm[32];
    int bx = blockIdx.x, src = 0;
    if (A.nb > 1) { src = bx & (A.nb - 1); bx >>= (31 - __clz(A.nb)); }   // grouped sources (nb = 2 | 4): see DslashArgs::nb
    A.in = (const char*)A.in + src * A.mul_in * A.fstride;
    A.out = (char*)A.out + src * A.mul_out * A.fstride;
    if (A.x) A.x = (const char*)A.x + src * A.mul_x * A.fstride;
    A.sc += src;
    A.partials += src * TM_PSTRIDE;
    if (guard_skip(A.sc, A.guard)) return;
    const Geom& g = A.g;
    const int h = bx * blockDim.x + threadIdx.x;
    double nrm = 0.0;
    if (h < g.Vh) {
        int xh, y, z, t;
        site_coords(g, h, xh, y, z, t);
        const int odd = (y + z + t + A.parity) & 1;     // x = 2*xh + odd
        const S* in = (const S*)A.in;
        const S* gauge = (const S*)A.gauge;
        F acc[24];
#pragma unroll
        for (int i = 0; i < 24; i++) acc[i] = 0;
        const F sf = -A.dsign, sb = A.dsign;           // forward: (1 - g), backward: (1 + g)
        const int row = h - xh;
        // x
        {
            const int xp = odd ? (xh + 1 == g.Xh ? 0 : xh + 1) : xh;
            const int xm = odd ? xh : (xh == 0 ? g.Xh - 1 : xh - 1);
            hop<0, 1, S, R>(in, gauge, g, A.parity, h, row + xp, sf, F(1), false, acc);
            hop<0, 0, S, R>(in, gauge, g, A.parity, h, row + xm, sb, F(1), false, acc);
        }
        // y
        {
            const int hp = (y + 1 == g.X1) ? h - (g.X1 - 1) * g.s1 : h + g.s1;
            const int hm = (y == 0) ? h + (g.X1 - 1) * g.s1 : h - g.s1;
            hop<1, 1, S, R>(in, gauge, g, A.parity, h, hp, sf, F(1), false, acc);
            hop<1, 0, S, R>(in, gauge, g, A.parity, h, hm, sb, F(1), false, acc);
        }
        // z
        {
            const int hp = (z + 1 == g.X2) ? h - (g.X2 - 1) * g.s2 : h + g.s2;
            const int hm = (z == 0) ? h + (g.X2 - 1) * g.s2 : h - g.s2;
            hop<2, 1, S, R>(in, gauge, g, A.parity, h, hp, sf, F(1), false, acc);
            hop<2, 0, S, R>(in, gauge, g, A.parity, h, hm, sb, F(1), false, acc);
        }
        // t (boundary sign when the hop wraps around)
        {
            const bool wp = (t + 1 == g.X3), wm = (t == 0);
            const int hp = wp ? h - (g.X3 - 1) * g.s3 : h + g.s3;
            const int hm = wm ? h + (g.X3 - 1) * g.s3 : h - g.s3;
            hop<3, 1, S, R>(in, gauge, g, A.parity, h, hp, sf, A.tb, wp, acc);
            hop<3, 0, S, R>(in, gauge, g, A.parity, h, hm, sb, A.tb, wm, acc);
        }
        // epilogue
#pragma unroll
        for (int i = 0; i < 24; i++) acc[i] *= A.c;
        if (A.xmode) {
            F xv[24];
            load_spinor<S>((const S*)A.x, g.Vh, h, xv);
            if (A.xmode == 2) {
#pragma unroll
                for (int i = 0; i < 12; i += 2) {       // upper: (1 + i a) x, lower: (1 - i a) x
                    acc[i] += xv[i] - A.a * xv[i + 1];
                    acc[i + 1] += xv[i + 1] + A.a * xv[i];
                    acc[12 + i] += xv[12 + i] + A.a * xv[12 + i + 1];
                    acc[12 + i + 1] += xv[12 + i + 1] - A.a * xv[12 + i];
                }
            } else {
#pragma unroll
                for (int i = 0; i < 24; i++) acc[i] += xv[i];
            }
        }
        if (A.post) {                                   // A^-1 = (1 - i a g5)/(1 + a^2)
            const F n = F(1) / (F(1) + A.a * A.a);
#pragma unroll
            for (int i = 0; i < 12; i += 2) {
                const F ur = acc[i], ui = acc[i + 1], lr = acc[12 + i], li = acc[12 + i + 1];
                acc[i] = n * (ur + A.a * ui);
                acc[i + 1] = n * (ui - A.a * ur);
                acc[12 + i] = n * (lr - A.a * li);
                acc[12 + i + 1] = n * (li + A.a * lr);
            }
        }
        store_spinor<S>((S*)A.out, g.Vh, h, acc);
        if (A.red_op != RED_NONE) {
#pragma unroll
            for (int i = 0; i < 24; i++) nrm += (double)acc[i] * (double)acc[i];
        }
    }
    if (A.red_op != RED_NONE) block_partial_at(nrm, A.partials, bx, sm);
}


// =====================================================================================================
// 16-bit storage path (fp16 / bf16), reconstruct-12 and -18.  Blackwell's mixed-precision FMA
// (PTX fma.rn.f32.f16 / .bf16 -> SASS FHFMA with .H0/.H1 operand selects) multiplies two 16-bit
// operands straight out of the packed registers and accumulates in fp32, so neither the links nor
// the neighbour spinors are ever unpacked: one 32-bit register = one complex number (re, im).
//   project     packed half2 arithmetic on the loaded spinor (result rounded to storage precision)
//   row 2       reconstruct-12: conj(row0 x row1) by FHFMA in fp32, packed back to 16 bit; reconstruct-18: loaded
//   SU(3) * u   FHFMA, fp32 accumulate
//   reconstruct   fp32, packed FADD2 / FFMA2 on (re, im) register pairs where the pairing allows
//   epilogue / norm   fp32 (as in the generic kernel)
//   links       the 8 links of a site are copied by cp.async into thread-private shared-memory slots at kernel
//               start (24 KB per CTA, 36 KB for reconstruct-18; no barrier: a thread reads only what it copied), so 2/3 of the kernel's
//               bytes are in flight without holding registers; spinors are register loads one hop ahead
template <typename S> struct Pk;
template <> struct Pk<__half> {
    typedef __half2 V2;
    template <int HA, int HB, int NEG> static __device__ __forceinline__ float fma(unsigned a, unsigned b, float c) {
        const unsigned short ah = HA ? (unsigned short)(a >> 16) : (unsigned short)(a & 0xffffu);
        const unsigned short bh = HB ? (unsigned short)(b >> 16) : (unsigned short)(b & 0xffffu);
        if (NEG) asm("{ .reg .b16 t; neg.f16 t, %1; fma.rn.f32.f16 %0, t, %2, %0; }" : "+f"(c) : "h"(ah), "h"(bh));
        else     asm("fma.rn.f32.f16 %0, %1, %2, %0;" : "+f"(c) : "h"(ah), "h"(bh));
        return c;
    }
    static __device__ __forceinline__ V2 make(float lo, float hi) { return __floats2half2_rn(lo, hi); }
};
template <> struct Pk<__nv_bfloat16> {
    typedef __nv_bfloat162 V2;
    template <int HA, int HB, int NEG> static __device__ __forceinline__ float fma(unsigned a, unsigned b, float c) {
        const unsigned short ah = HA ? (unsigned short)(a >> 16) : (unsigned short)(a & 0xffffu);
        const unsigned short bh = HB ? (unsigned short)(b >> 16) : (unsigned short)(b & 0xffffu);
        if (NEG) asm("{ .reg .b16 t; neg.bf16 t, %1; fma.rn.f32.bf16 %0, t, %2, %0; }" : "+f"(c) : "h"(ah), "h"(bh));
        else     asm("fma.rn.f32.bf16 %0, %1, %2, %0;" : "+f"(c) : "h"(ah), "h"(bh));
        return c;
    }
    static __device__ __forceinline__ V2 make(float lo, float hi) { return __floats2bfloat162_rn(lo, hi); }
};
template <typename V2> __device__ __forceinline__ V2 as_v2(unsigned w) { return *reinterpret_cast<V2*>(&w); }
template <typename V2> __device__ __forceinline__ unsigned as_u(V2 v) { return *reinterpret_cast<unsigned*>(&v); }

// acc += (CONJ ? conj(a) : a) * b for packed complex a, b
template <typename S, int CONJ>
__device__ __forceinline__ void cmadd16(unsigned a, unsigned b, float& re, float& im) {
    re = Pk<S>::template fma<0, 0, 0>(a, b, re);
    re = Pk<S>::template fma<1, 1, CONJ ? 0 : 1>(a, b, re);
    im = Pk<S>::template fma<0, 1, 0>(a, b, im);
    im = Pk<S>::template fma<1, 0, CONJ ? 1 : 0>(a, b, im);
}

// packed half-spinor u[sp*3 + c] = psi_up + s * B_mu psi_low, s = SGN (compile time)
template <int MU, int SGN, typename S>
__device__ __forceinline__ void project16(const unsigned* p, unsigned* u) {
    typedef typename Pk<S>::V2 V2;
    const V2 mi = Pk<S>::make((float)SGN, (float)-SGN);      // multiply by -i*s after a (re,im) swap
    const V2 pi = Pk<S>::make((float)-SGN, (float)SGN);      // multiply by +i*s after a swap
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const V2 p0 = as_v2<V2>(p[c]), p1 = as_v2<V2>(p[3 + c]), p2 = as_v2<V2>(p[6 + c]), p3 = as_v2<V2>(p[9 + c]);
        V2 u0, u1;
        if (MU == 0) {          // (-i psi3, -i psi2)
            u0 = __hfma2(__lowhigh2highlow(p3), mi, p0);
            u1 = __hfma2(__lowhigh2highlow(p2), mi, p1);
        } else if (MU == 1) {   // (-psi3, psi2)
            u0 = SGN > 0 ? __hsub2(p0, p3) : __hadd2(p0, p3);
            u1 = SGN > 0 ? __hadd2(p1, p2) : __hsub2(p1, p2);
        } else if (MU == 2) {   // (-i psi2, i psi3)
            u0 = __hfma2(__lowhigh2highlow(p2), mi, p0);
            u1 = __hfma2(__lowhigh2highlow(p3), pi, p1);
        } else {                // (psi2, psi3)
            u0 = SGN > 0 ? __hadd2(p0, p2) : __hsub2(p0, p2);
            u1 = SGN > 0 ? __hadd2(p1, p3) : __hsub2(p1, p3);
        }
        u[c] = as_u(u0);
        u[3 + c] = as_u(u1);
    }
}

// stage_link16: the link of one hop copied into the thread's private shared-memory slots with cp.async (no
// registers held while the copy is in flight); slot k * 128 of the thread's column, k = 0..2
// Link storage of the 16-bit copies (common.cuh GaugeLayout): reconstruct-12 = 3 chunks of 8 bytes (two complex
// numbers each), reconstruct-18 = 9 chunks of 4 bytes (one complex number each); LinkSlot<R>::T is one chunk.
template <int R> struct LinkSlot;
template <> struct LinkSlot<12> { typedef uint2 T; static constexpr int NCH = 3; };
template <> struct LinkSlot<18> { typedef unsigned T; static constexpr int NCH = 9; };

template <int MU, int FWD, typename S, int R>
__device__ __forceinline__ void stage_link16(const S* gauge, size_t Vh, int par_out, size_t h_out, size_t h_nb,
                                             typename LinkSlot<R>::T* slot) {
    typedef typename LinkSlot<R>::T C;
    constexpr int NCH = LinkSlot<R>::NCH;
    const size_t hl = FWD ? h_out : h_nb;
    const int pl = FWD ? par_out : 1 - par_out;
    const unsigned gi = (unsigned)(pl * 4 + MU) * (unsigned)NCH * (unsigned)Vh + (unsigned)hl;
    const C* g = reinterpret_cast<const C*>(gauge);
#pragma unroll
    for (int k = 0; k < NCH; k++) {
        const unsigned dst = (unsigned)__cvta_generic_to_shared(slot + k * 128);
        asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(dst), "l"(g + (gi + (unsigned)k * (unsigned)Vh)), "n"(sizeof(C)) : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
}
template <int N> __device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
template <typename S>
__device__ __forceinline__ void load_spinor16(const S* in, size_t Vh, size_t h_nb, unsigned* p) {
    const uint4* f = reinterpret_cast<const uint4*>(in) + h_nb;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const uint4 q = __ldg(f + (size_t)k * Vh);
        p[4 * k] = q.x; p[4 * k + 1] = q.y; p[4 * k + 2] = q.z; p[4 * k + 3] = q.w;
    }
}
__device__ __forceinline__ void read_link16(const uint2* slot, unsigned* U) {
#pragma unroll
    for (int k = 0; k < 3; k++) { const uint2 q = slot[k * 128]; U[2 * k] = q.x; U[2 * k + 1] = q.y; }
}
__device__ __forceinline__ void read_link16(const unsigned* slot, unsigned* U) {
#pragma unroll
    for (int k = 0; k < 9; k++) U[k] = slot[k * 128];
}

template <int MU, int FWD, typename S, int R>
__device__ __forceinline__ void load16(const S* in, const S* gauge, size_t Vh, int par_out, size_t h_out, size_t h_nb,
                                       unsigned* p, unsigned* U) {
    const uint4* f = reinterpret_cast<const uint4*>(in) + h_nb;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const uint4 q = __ldg(f + (size_t)k * Vh);
        p[4 * k] = q.x; p[4 * k + 1] = q.y; p[4 * k + 2] = q.z; p[4 * k + 3] = q.w;
    }
    const size_t hl = FWD ? h_out : h_nb;
    const int pl = FWD ? par_out : 1 - par_out;
    // 32-bit element index (8 * 9 * Vh < 2^31 for every supported lattice): one IMAD.WIDE per load
    const unsigned gi = (unsigned)(pl * 4 + MU) * (unsigned)LinkSlot<R>::NCH * (unsigned)Vh + (unsigned)hl;
    if (R == 12) {
        const uint2* g = reinterpret_cast<const uint2*>(gauge);
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const uint2 q = __ldcs(g + (gi + (unsigned)k * (unsigned)Vh));
            U[2 * k] = q.x; U[2 * k + 1] = q.y;
        }
    } else {
        const unsigned* g = reinterpret_cast<const unsigned*>(gauge);
#pragma unroll
        for (int k = 0; k < 9; k++) U[k] = __ldcs(g + (gi + (unsigned)k * (unsigned)Vh));
    }
}

// packed fp32 pair arithmetic (Blackwell FADD2 / FFMA2): acc pairs (re, im) live in aligned register pairs
__device__ __forceinline__ void add2(float& ar, float& ai, float br, float bi) {
    unsigned long long a, b;
    asm("mov.b64 %0, {%1, %2};" : "=l"(a) : "f"(ar), "f"(ai));
    asm("mov.b64 %0, {%1, %2};" : "=l"(b) : "f"(br), "f"(bi));
    asm("add.rn.f32x2 %0, %0, %1;" : "+l"(a) : "l"(b));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(ar), "=f"(ai) : "l"(a));
}
__device__ __forceinline__ void sub2(float& ar, float& ai, float br, float bi) {
    unsigned long long a, b, m;
    asm("mov.b64 %0, {%1, %2};" : "=l"(a) : "f"(ar), "f"(ai));
    asm("mov.b64 %0, {%1, %2};" : "=l"(b) : "f"(br), "f"(bi));
    asm("mov.b64 %0, {%1, %1};" : "=l"(m) : "f"(-1.f));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(a) : "l"(b), "l"(m));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(ar), "=f"(ai) : "l"(a));
}

// acc_up += v ; acc_low += s * B_mu^dag v  (s = +-1 at compile time), packed where the pairing allows
template <int MU, int SGN>
__device__ __forceinline__ void reconstruct16(const float* v, float* acc) {
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const float v0r = v[2 * c], v0i = v[2 * c + 1], v1r = v[6 + 2 * c], v1i = v[6 + 2 * c + 1];
        add2(acc[2 * c], acc[2 * c + 1], v0r, v0i);
        add2(acc[6 + 2 * c], acc[6 + 2 * c + 1], v1r, v1i);
        if (MU == 0) {          // B^dag v = (i v1, i v0)
            if (SGN > 0) { acc[12 + 2 * c] -= v1i; acc[12 + 2 * c + 1] += v1r; acc[18 + 2 * c] -= v0i; acc[18 + 2 * c + 1] += v0r; }
            else         { acc[12 + 2 * c] += v1i; acc[12 + 2 * c + 1] -= v1r; acc[18 + 2 * c] += v0i; acc[18 + 2 * c + 1] -= v0r; }
        } else if (MU == 1) {   // (v1, -v0)
            if (SGN > 0) { add2(acc[12 + 2 * c], acc[12 + 2 * c + 1], v1r, v1i); sub2(acc[18 + 2 * c], acc[18 + 2 * c + 1], v0r, v0i); }
            else         { sub2(acc[12 + 2 * c], acc[12 + 2 * c + 1], v1r, v1i); add2(acc[18 + 2 * c], acc[18 + 2 * c + 1], v0r, v0i); }
        } else if (MU == 2) {   // (i v0, -i v1)
            if (SGN > 0) { acc[12 + 2 * c] -= v0i; acc[12 + 2 * c + 1] += v0r; acc[18 + 2 * c] += v1i; acc[18 + 2 * c + 1] -= v1r; }
            else         { acc[12 + 2 * c] += v0i; acc[12 + 2 * c + 1] -= v0r; acc[18 + 2 * c] -= v1i; acc[18 + 2 * c + 1] += v1r; }
        } else {                // (v0, v1)
            if (SGN > 0) { add2(acc[12 + 2 * c], acc[12 + 2 * c + 1], v0r, v0i); add2(acc[18 + 2 * c], acc[18 + 2 * c + 1], v1r, v1i); }
            else         { sub2(acc[12 + 2 * c], acc[12 + 2 * c + 1], v0r, v0i); sub2(acc[18 + 2 * c], acc[18 + 2 * c + 1], v1r, v1i); }
        }
    }
}

template <int MU, int FWD, int DAGGER, typename S, int R>
__device__ __forceinline__ void compute16(const unsigned* p, const unsigned* Uin, float bsign, bool wrap, float* acc,
                                          unsigned* row2 = nullptr /* R == 12: receives the rebuilt third row */) {
    typedef typename Pk<S>::V2 V2;
    constexpr int SGN = (FWD ? -1 : 1) * (DAGGER ? -1 : 1);       // forward: (1 - g), backward: (1 + g)
    unsigned U[9], u[6];
#pragma unroll
    for (int i = 0; i < R / 2; i++) U[i] = Uin[i];
    project16<MU, SGN, S>(p, u);
    if (MU == 3 && wrap) {
        const V2 b2 = Pk<S>::make(bsign, bsign);
#pragma unroll
        for (int i = 0; i < 6; i++) u[i] = as_u(__hmul2(as_v2<V2>(u[i]), b2));
    }
    // row 2 = conj(row0 x row1) = conj(a_i b_j - a_j b_i): one FHFMA chain per real (negation is an operand modifier)
#pragma unroll
    for (int c = 0; c < (R == 12 ? 3 : 0); c++) {
        const int i = (c + 1) % 3, j = (c + 2) % 3;
        float re = 0.f, nim = 0.f;
        re  = Pk<S>::template fma<0, 0, 0>(U[i], U[3 + j], re);
        nim = Pk<S>::template fma<0, 1, 1>(U[i], U[3 + j], nim);
        re  = Pk<S>::template fma<1, 1, 1>(U[i], U[3 + j], re);
        nim = Pk<S>::template fma<1, 0, 1>(U[i], U[3 + j], nim);
        re  = Pk<S>::template fma<0, 0, 1>(U[j], U[3 + i], re);
        nim = Pk<S>::template fma<0, 1, 0>(U[j], U[3 + i], nim);
        re  = Pk<S>::template fma<1, 1, 0>(U[j], U[3 + i], re);
        nim = Pk<S>::template fma<1, 0, 0>(U[j], U[3 + i], nim);
        U[6 + c] = as_u(Pk<S>::make(re, nim));
    }
    if (R == 12 && row2) { row2[0] = U[6]; row2[1] = U[7]; row2[2] = U[8]; }
    // v = U u (or U^dag u) accumulated straight into the upper components of acc; the lower components
    // get s B_mu^dag v from the increment (new - old)
    float v[12];
#pragma unroll
    for (int sp = 0; sp < 2; sp++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            float re = 0.f, im = 0.f;
#pragma unroll
            for (int b = 0; b < 3; b++) {
                if (FWD) cmadd16<S, 0>(U[a * 3 + b], u[sp * 3 + b], re, im);       // U u
                else     cmadd16<S, 1>(U[b * 3 + a], u[sp * 3 + b], re, im);       // U^dag u
            }
            v[sp * 6 + 2 * a] = re;
            v[sp * 6 + 2 * a + 1] = im;
        }
    reconstruct16<MU, SGN>(v, acc);
}

// epilogue of the 16-bit kernels for one site: res = c * acc (+ x | + A x), optional A^-1, store, optional |res|^2
template <typename S>
__device__ __forceinline__ void dslash16_epilogue(const DslashArgs<float>& A, const S* xop, S* out, const Geom& g, int h,
                                                  float* acc, double& nrm) {
    // epilogue: res = c * acc (+ x | + A x), optional A^-1, store, optional norm
    const float cf = A.c, a = A.a;
    if (A.xmode) {
        float xv[24];
        load_spinor<S>(xop, g.Vh, h, xv);
        if (A.xmode == 2) {
#pragma unroll
            for (int i = 0; i < 12; i += 2) {
                float t0 = xv[i]; t0 -= a * xv[i + 1];              acc[i] = fmaf(cf, acc[i], t0);
                float t1 = xv[i + 1]; t1 += a * xv[i];              acc[i + 1] = fmaf(cf, acc[i + 1], t1);
                float t2 = xv[12 + i]; t2 += a * xv[12 + i + 1];    acc[12 + i] = fmaf(cf, acc[12 + i], t2);
                float t3 = xv[12 + i + 1]; t3 -= a * xv[12 + i];    acc[12 + i + 1] = fmaf(cf, acc[12 + i + 1], t3);
            }
        } else {
#pragma unroll
            for (int i = 0; i < 24; i++) acc[i] = fmaf(cf, acc[i], xv[i]);
        }
    } else {
#pragma unroll
        for (int i = 0; i < 24; i++) acc[i] *= cf;
    }
    if (A.post) {
        const float n = 1.f / (1.f + a * a);
#pragma unroll
        for (int i = 0; i < 12; i += 2) {
            const float ur = acc[i], ui = acc[i + 1], lr = acc[12 + i], li = acc[12 + i + 1];
            acc[i] = n * (ur + a * ui);
            acc[i + 1] = n * (ui - a * ur);
            acc[12 + i] = n * (lr - a * li);
            acc[12 + i + 1] = n * (li + a * lr);
        }
    }
    store_spinor<S>(out, g.Vh, h, acc);
    if (A.red_op != RED_NONE) {
        float n2 = 0.f;      // 24 terms in fp32, then fp64 across sites
#pragma unroll
        for (int i = 0; i < 24; i++) n2 = fmaf(acc[i], acc[i], n2);
        nrm = (double)n2;
    }
}

template <typename S, int DAGGER, int PIPE, int MINB, int R>
__global__ void __launch_bounds__(128, MINB) dslash16_kernel(DslashArgs<float> A) {
    __shared__ double sm[32];
    int bx = blockIdx.x, src = 0;
    if (A.nb > 1) { src = bx & (A.nb - 1); bx >>= (31 - __clz(A.nb)); }
    A.in = (const char*)A.in + src * A.mul_in * A.fstride;
    A.out = (char*)A.out + src * A.mul_out * A.fstride;
    if (A.x) A.x = (const char*)A.x + src * A.mul_x * A.fstride;
    A.sc += src;
    A.partials += src * TM_PSTRIDE;
    if (guard_skip(A.sc, A.guard)) return;
    const Geom& g = A.g;
    const int h = bx * blockDim.x + threadIdx.x;
    double nrm = 0.0;
    if (h < g.Vh) {
        int xh, y, z, t;
        site_coords(g, h, xh, y, z, t);
        const int odd = (y + z + t + A.parity) & 1;
        const S* in = (const S*)A.in;
        const S* gauge = (const S*)A.gauge;
        const size_t Vh = g.Vh;
        float acc[24];
#pragma unroll
        for (int i = 0; i < 24; i++) acc[i] = 0.f;
        const int row = h - xh;
        const int xp = row + (odd ? (xh + 1 == g.Xh ? 0 : xh + 1) : xh);
        const int xm = row + (odd ? xh : (xh == 0 ? g.Xh - 1 : xh - 1));
        const int yp = (y + 1 == g.X1) ? h - (g.X1 - 1) * g.s1 : h + g.s1;
        const int ym = (y == 0) ? h + (g.X1 - 1) * g.s1 : h - g.s1;
        const int zp = (z + 1 == g.X2) ? h - (g.X2 - 1) * g.s2 : h + g.s2;
        const int zm = (z == 0) ? h + (g.X2 - 1) * g.s2 : h - g.s2;
        const bool wp = (t + 1 == g.X3), wm = (t == 0);
        const int tp = wp ? h - (g.X3 - 1) * g.s3 : h + g.s3;
        const int tm = wm ? h + (g.X3 - 1) * g.s3 : h - g.s3;
        const int par = A.parity;
        if (A.xmode) {              // the epilogue's x operand: into L2 now (see dslash16_group_kernel)
            const uint4* xf = reinterpret_cast<const uint4*>(A.x) + h;
#pragma unroll
            for (int k = 0; k < 3; k++) asm volatile("prefetch.global.L2 [%0];" ::"l"(xf + (size_t)k * Vh));
        }
        unsigned pa[12], ua[R / 2];
        constexpr int LS = LinkSlot<R>::NCH * 128;             // slots of one hop
        if (PIPE == 2) {
            // links: all 8 hops staged by cp.async up front (thread-private slots, no barrier needed);
            // spinors: register loads one hop ahead
            __shared__ typename LinkSlot<R>::T smg[8 * LS];
            typename LinkSlot<R>::T* sl = smg + threadIdx.x;
            stage_link16<0, 1, S, R>(gauge, Vh, par, h, xp, sl + 0 * LS);
            stage_link16<0, 0, S, R>(gauge, Vh, par, h, xm, sl + 1 * LS);
            stage_link16<1, 1, S, R>(gauge, Vh, par, h, yp, sl + 2 * LS);
            stage_link16<1, 0, S, R>(gauge, Vh, par, h, ym, sl + 3 * LS);
            stage_link16<2, 1, S, R>(gauge, Vh, par, h, zp, sl + 4 * LS);
            stage_link16<2, 0, S, R>(gauge, Vh, par, h, zm, sl + 5 * LS);
            stage_link16<3, 1, S, R>(gauge, Vh, par, h, tp, sl + 6 * LS);
            stage_link16<3, 0, S, R>(gauge, Vh, par, h, tm, sl + 7 * LS);
            unsigned pb[12];
            load_spinor16<S>(in, Vh, xp, pa);
            load_spinor16<S>(in, Vh, xm, pb);
            cp_wait<7>(); read_link16(sl + 0 * LS, ua); compute16<0, 1, DAGGER, S, R>(pa, ua, 1.f, false, acc);
            load_spinor16<S>(in, Vh, yp, pa);
            cp_wait<6>(); read_link16(sl + 1 * LS, ua); compute16<0, 0, DAGGER, S, R>(pb, ua, 1.f, false, acc);
            load_spinor16<S>(in, Vh, ym, pb);
            cp_wait<5>(); read_link16(sl + 2 * LS, ua); compute16<1, 1, DAGGER, S, R>(pa, ua, 1.f, false, acc);
            load_spinor16<S>(in, Vh, zp, pa);
            cp_wait<4>(); read_link16(sl + 3 * LS, ua); compute16<1, 0, DAGGER, S, R>(pb, ua, 1.f, false, acc);
            load_spinor16<S>(in, Vh, zm, pb);
            cp_wait<3>(); read_link16(sl + 4 * LS, ua); compute16<2, 1, DAGGER, S, R>(pa, ua, 1.f, false, acc);
            load_spinor16<S>(in, Vh, tp, pa);
            cp_wait<2>(); read_link16(sl + 5 * LS, ua); compute16<2, 0, DAGGER, S, R>(pb, ua, 1.f, false, acc);
            load_spinor16<S>(in, Vh, tm, pb);
            cp_wait<1>(); read_link16(sl + 6 * LS, ua); compute16<3, 1, DAGGER, S, R>(pa, ua, A.tb, wp, acc);
            cp_wait<0>(); read_link16(sl + 7 * LS, ua); compute16<3, 0, DAGGER, S, R>(pb, ua, A.tb, wm, acc);
        } else {
            load16<0, 1, S, R>(in, gauge, Vh, par, h, xp, pa, ua); compute16<0, 1, DAGGER, S, R>(pa, ua, 1.f, false, acc);
            load16<0, 0, S, R>(in, gauge, Vh, par, h, xm, pa, ua); compute16<0, 0, DAGGER, S, R>(pa, ua, 1.f, false, acc);
            load16<1, 1, S, R>(in, gauge, Vh, par, h, yp, pa, ua); compute16<1, 1, DAGGER, S, R>(pa, ua, 1.f, false, acc);
            load16<1, 0, S, R>(in, gauge, Vh, par, h, ym, pa, ua); compute16<1, 0, DAGGER, S, R>(pa, ua, 1.f, false, acc);
            load16<2, 1, S, R>(in, gauge, Vh, par, h, zp, pa, ua); compute16<2, 1, DAGGER, S, R>(pa, ua, 1.f, false, acc);
            load16<2, 0, S, R>(in, gauge, Vh, par, h, zm, pa, ua); compute16<2, 0, DAGGER, S, R>(pa, ua, 1.f, false, acc);
            load16<3, 1, S, R>(in, gauge, Vh, par, h, tp, pa, ua); compute16<3, 1, DAGGER, S, R>(pa, ua, A.tb, wp, acc);
            load16<3, 0, S, R>(in, gauge, Vh, par, h, tm, pa, ua); compute16<3, 0, DAGGER, S, R>(pa, ua, A.tb, wm, acc);
        }
        dslash16_epilogue<S>(A, (const S*)A.x, (S*)A.out, g, h, acc, nrm);
    }
    if (A.red_op != RED_NONE) block_partial_at(nrm, A.partials, bx, sm);
}

// -----------------------------------------------------------------------------------------------------
// Grouped launches (tm_dslash_multi, the solver's launch shape): one CTA applies the stencil to the same 128 sites
// of `ns` sources, one after the other.  What depends only on the sites is then done once per CTA instead of once
// per source: the site / neighbour / link index arithmetic, the 24 cp.async of the links, and the rebuild of the
// third link row -- the first source that runs writes the rebuilt rows next to the staged ones (thread-private
// slots: no barrier), the others read complete links.  Same arithmetic in the same order per source: results are
// bit-identical to one source per CTA.  (reconstruct-12 only.)
#define D16G_CH 4            // 8-byte chunks per hop and thread: rows 0, 1 as staged (3) + two thirds of the rebuilt row 2;
                             // its last complex number sits in a 4-byte array of its own: 36 KB of slots per CTA, so that
                             // 5 CTAs stay below the 196 KB shared-memory carve-out (at 228 KB the 28 KB left for L1 cost 21 %)

template <typename S, int DAGGER, int FIRST>
__device__ __forceinline__ void hops16_group(const S* in, size_t Vh, uint2* sl, unsigned* sl1, const int* nbr, float tb, bool wp,
                                             bool wm, float* acc) {
    constexpr int LS = D16G_CH * 128;
    unsigned pa[12], pb[12], ua[9], row2[3];
    auto link = [&](int j) {
        const uint2* s = sl + j * LS;
        const uint2 q0 = s[0], q1 = s[128], q2 = s[256];
        ua[0] = q0.x; ua[1] = q0.y; ua[2] = q1.x; ua[3] = q1.y; ua[4] = q2.x; ua[5] = q2.y;
        if (!FIRST) { const uint2 q3 = s[384]; ua[6] = q3.x; ua[7] = q3.y; ua[8] = sl1[j * 128]; }
    };
    auto keep = [&](int j) {
        if (FIRST) { sl[j * LS + 384] = make_uint2(row2[0], row2[1]); sl1[j * 128] = row2[2]; }
    };
#define D16G_HOP(J, MU, FWD, PBUF, BS, WR)                                                                    \
    do {                                                                                                       \
        if (FIRST) cp_wait<7 - (J)>();                                                                         \
        link(J);                                                                                               \
        if (FIRST) { compute16<MU, FWD, DAGGER, S, 12>(PBUF, ua, BS, WR, acc, row2); keep(J); }                 \
        else compute16<MU, FWD, DAGGER, S, 18>(PBUF, ua, BS, WR, acc);                                         \
    } while (0)
    load_spinor16<S>(in, Vh, nbr[0], pa);
    load_spinor16<S>(in, Vh, nbr[1], pb);
    D16G_HOP(0, 0, 1, pa, 1.f, false);
    load_spinor16<S>(in, Vh, nbr[2], pa);
    D16G_HOP(1, 0, 0, pb, 1.f, false);
    load_spinor16<S>(in, Vh, nbr[3], pb);
    D16G_HOP(2, 1, 1, pa, 1.f, false);
    load_spinor16<S>(in, Vh, nbr[4], pa);
    D16G_HOP(3, 1, 0, pb, 1.f, false);
    load_spinor16<S>(in, Vh, nbr[5], pb);
    D16G_HOP(4, 2, 1, pa, 1.f, false);
    load_spinor16<S>(in, Vh, nbr[6], pa);
    D16G_HOP(5, 2, 0, pb, 1.f, false);
    load_spinor16<S>(in, Vh, nbr[7], pb);
    D16G_HOP(6, 3, 1, pa, tb, wp);
    D16G_HOP(7, 3, 0, pb, tb, wm);
#undef D16G_HOP
}

template <typename S, int DAGGER, int MINB>
__global__ void __launch_bounds__(128, MINB) dslash16_group_kernel(DslashArgs<float> A) {
    __shared__ double sm[32];
    __shared__ uint2 smg[8 * D16G_CH * 128];
    __shared__ unsigned smg1[8 * 128];
    // CTA index = (tile, group of ns sources): the nb / ns CTAs of a tile are neighbours, so the links they all stage
    // cross HBM once (L2); ns and nb are powers of two
    const int ns = A.ns, ng = A.nb / ns;
    const int bx = blockIdx.x / ng, src0 = (blockIdx.x - bx * ng) * ns;
    const Geom& g = A.g;
    const int h = bx * blockDim.x + threadIdx.x;
    const bool live = h < g.Vh;
    const S* gauge = (const S*)A.gauge;
    const size_t Vh = g.Vh;
    const int par = A.parity;
    uint2* sl = smg + threadIdx.x;
    unsigned* sl1 = smg1 + threadIdx.x;
    int nbr[8];
    bool wp = false, wm = false;
    if (live) {
        int xh, y, z, t;
        site_coords(g, h, xh, y, z, t);
        const int odd = (y + z + t + par) & 1;
        const int row = h - xh;
        nbr[0] = row + (odd ? (xh + 1 == g.Xh ? 0 : xh + 1) : xh);
        nbr[1] = row + (odd ? xh : (xh == 0 ? g.Xh - 1 : xh - 1));
        nbr[2] = (y + 1 == g.X1) ? h - (g.X1 - 1) * g.s1 : h + g.s1;
        nbr[3] = (y == 0) ? h + (g.X1 - 1) * g.s1 : h - g.s1;
        nbr[4] = (z + 1 == g.X2) ? h - (g.X2 - 1) * g.s2 : h + g.s2;
        nbr[5] = (z == 0) ? h + (g.X2 - 1) * g.s2 : h - g.s2;
        wp = (t + 1 == g.X3); wm = (t == 0);
        nbr[6] = wp ? h - (g.X3 - 1) * g.s3 : h + g.s3;
        nbr[7] = wm ? h + (g.X3 - 1) * g.s3 : h - g.s3;
        constexpr int LS = D16G_CH * 128;
        stage_link16<0, 1, S, 12>(gauge, Vh, par, h, nbr[0], sl + 0 * LS);
        stage_link16<0, 0, S, 12>(gauge, Vh, par, h, nbr[1], sl + 1 * LS);
        stage_link16<1, 1, S, 12>(gauge, Vh, par, h, nbr[2], sl + 2 * LS);
        stage_link16<1, 0, S, 12>(gauge, Vh, par, h, nbr[3], sl + 3 * LS);
        stage_link16<2, 1, S, 12>(gauge, Vh, par, h, nbr[4], sl + 4 * LS);
        stage_link16<2, 0, S, 12>(gauge, Vh, par, h, nbr[5], sl + 5 * LS);
        stage_link16<3, 1, S, 12>(gauge, Vh, par, h, nbr[6], sl + 6 * LS);
        stage_link16<3, 0, S, 12>(gauge, Vh, par, h, nbr[7], sl + 7 * LS);
    }
    bool first = true;                         // no source has used (and completed) the staged links yet
    for (int si = 0; si < ns; si++) {
        const int src = src0 + si;
        if (guard_skip(A.sc + src, A.guard)) continue;            // uniform over the CTA
        const S* in = (const S*)((const char*)A.in + (size_t)src * A.mul_in * A.fstride);
        S* out = (S*)((char*)A.out + (size_t)src * A.mul_out * A.fstride);
        const S* xop = A.x ? (const S*)((const char*)A.x + (size_t)src * A.mul_x * A.fstride) : nullptr;
        double nrm = 0.0;
        if (live) {
            float acc[24];
#pragma unroll
            for (int i = 0; i < 24; i++) acc[i] = 0.f;
            if (A.xmode) {          // the epilogue's x operand is a load nothing hides (no registers to issue it early): pull it into L2
                                    // now (392.5 -> 376.5 us per 8-source launch; prefetching the next source's first neighbours too: no gain)
                const uint4* xf = reinterpret_cast<const uint4*>(xop) + h;
#pragma unroll
                for (int k = 0; k < 3; k++) asm volatile("prefetch.global.L2 [%0];" ::"l"(xf + (size_t)k * Vh));
            }
            if (first) hops16_group<S, DAGGER, 1>(in, Vh, sl, sl1, nbr, A.tb, wp, wm, acc);
            else       hops16_group<S, DAGGER, 0>(in, Vh, sl, sl1, nbr, A.tb, wp, wm, acc);
            dslash16_epilogue<S>(A, xop, out, g, h, acc, nrm);
        }
        first = false;
        if (A.red_op != RED_NONE) block_partial_at(nrm, A.partials + (size_t)src * TM_PSTRIDE, bx, sm);
    }
}

// =====================================================================================================
// fp32 storage, reconstruct-12, packed arithmetic: one complex number per 64-bit register pair, Blackwell FFMA2 /
// FADD2 (fma.rn.f32x2 with a broadcast real scalar: one issue slot per complex-times-real FMA).  Same mathematics
// and data layout as dslash_kernel<float, 12>; ~20 % fewer instructions per site (the grouped launches of this
// kernel are bound by instruction issue and board power, not by HBM).
typedef P2<float>::T c2;     // (re, im)

template <int MU, int FWD, int DAGGER>
__device__ __forceinline__ void hop32(const float* in, const float* gauge, size_t Vh, int par_out, size_t h_out,
                                      size_t h_nb, float bsign, bool wrap, c2* acc) {
    constexpr float SGN = (float)((FWD ? -1 : 1) * (DAGGER ? -1 : 1));      // forward: (1 - g), backward: (1 + g)
    c2 p[12];
    {
        // 32-bit element indices (24 * Vh < 2^31 for every supported lattice): one IMAD.WIDE per load instead of a
        // 64-bit add
        const float4* f = reinterpret_cast<const float4*>(in);
        const unsigned hn = (unsigned)h_nb, vh = (unsigned)Vh;
#pragma unroll
        for (int k = 0; k < 6; k++) {
            const float4 q = __ldg(f + (hn + (unsigned)k * vh));
            p[2 * k] = P2<float>::make(q.x, q.y);
            p[2 * k + 1] = P2<float>::make(q.z, q.w);
        }
    }
    float U[18];
    {
        const size_t hl = FWD ? h_out : h_nb;
        const int pl = FWD ? par_out : 1 - par_out;
        const float4* g = reinterpret_cast<const float4*>(gauge);
        const unsigned gi = (unsigned)(pl * 4 + MU) * 3u * (unsigned)Vh + (unsigned)hl;
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const float4 q = __ldcs(g + (gi + (unsigned)k * (unsigned)Vh));
            U[4 * k] = q.x; U[4 * k + 1] = q.y; U[4 * k + 2] = q.z; U[4 * k + 3] = q.w;
        }
#pragma unroll
        for (int c = 0; c < 3; c++) {          // row 2 = conj(row0 x row1)
            const int i = (c + 1) % 3, j = (c + 2) % 3;
            const float ar = U[2 * i], ai = U[2 * i + 1], br = U[6 + 2 * j], bi = U[6 + 2 * j + 1];
            const float cr = U[2 * j], ci = U[2 * j + 1], dr = U[6 + 2 * i], di = U[6 + 2 * i + 1];
            float re = ar * br; re -= ai * bi; re -= cr * dr; re += ci * di;
            float im = ar * bi; im += ai * br; im -= cr * di; im -= ci * dr;
            U[12 + 2 * c] = re;
            U[12 + 2 * c + 1] = -im;
        }
    }
    // half-spinor u = psi_up + s B_mu psi_low (B_x = -i s_x, B_y = -i s_y, B_z = -i s_z, B_t = 1)
    c2 u[6];
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const c2 p0 = p[c], p1 = p[3 + c], p2 = p[6 + c], p3 = p[9 + c];
        if (MU == 0) {          // (-i psi3, -i psi2)
            u[c] = P2<float>::fma_si(-SGN, p3, p0);
            u[3 + c] = P2<float>::fma_si(-SGN, p2, p1);
        } else if (MU == 1) {   // (-psi3, psi2)
            u[c] = P2<float>::fma_s(-SGN, p3, p0);
            u[3 + c] = P2<float>::fma_s(SGN, p2, p1);
        } else if (MU == 2) {   // (-i psi2, i psi3)
            u[c] = P2<float>::fma_si(-SGN, p2, p0);
            u[3 + c] = P2<float>::fma_si(SGN, p3, p1);
        } else {                // (psi2, psi3)
            u[c] = P2<float>::fma_s(SGN, p2, p0);
            u[3 + c] = P2<float>::fma_s(SGN, p3, p1);
        }
    }
    if (MU == 3 && wrap) {
#pragma unroll
        for (int i = 0; i < 6; i++) u[i] = P2<float>::mul_s(bsign, u[i]);
    }
    // v = U u (forward) or U^dag u (backward): (ur + i ui) x = ur x + ui (i x), accumulators updated round-robin
    c2 v[6];
#pragma unroll
    for (int i = 0; i < 6; i++) v[i] = P2<float>::make(0.f, 0.f);
#pragma unroll
    for (int b = 0; b < 3; b++) {
        float ur[3], ui[3];
#pragma unroll
        for (int a = 0; a < 3; a++) {
            ur[a] = FWD ? U[(a * 3 + b) * 2] : U[(b * 3 + a) * 2];
            ui[a] = FWD ? U[(a * 3 + b) * 2 + 1] : -U[(b * 3 + a) * 2 + 1];
        }
#pragma unroll
        for (int a = 0; a < 3; a++) {
            v[a] = P2<float>::fma_s(ur[a], u[b], v[a]);
            v[3 + a] = P2<float>::fma_s(ur[a], u[3 + b], v[3 + a]);
        }
#pragma unroll
        for (int a = 0; a < 3; a++) {
            v[a] = P2<float>::fma_si(ui[a], u[b], v[a]);
            v[3 + a] = P2<float>::fma_si(ui[a], u[3 + b], v[3 + a]);
        }
    }
    // acc_up += v ; acc_low += s B_mu^dag v
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const c2 v0 = v[c], v1 = v[3 + c];
        acc[c] = P2<float>::add(acc[c], v0);
        acc[3 + c] = P2<float>::add(acc[3 + c], v1);
        if (MU == 0) {          // (i v1, i v0)
            acc[6 + c] = P2<float>::fma_si(SGN, v1, acc[6 + c]);
            acc[9 + c] = P2<float>::fma_si(SGN, v0, acc[9 + c]);
        } else if (MU == 1) {   // (v1, -v0)
            acc[6 + c] = P2<float>::fma_s(SGN, v1, acc[6 + c]);
            acc[9 + c] = P2<float>::fma_s(-SGN, v0, acc[9 + c]);
        } else if (MU == 2) {   // (i v0, -i v1)
            acc[6 + c] = P2<float>::fma_si(SGN, v0, acc[6 + c]);
            acc[9 + c] = P2<float>::fma_si(-SGN, v1, acc[9 + c]);
        } else {                // (v0, v1)
            acc[6 + c] = P2<float>::fma_s(SGN, v0, acc[6 + c]);
            acc[9 + c] = P2<float>::fma_s(SGN, v1, acc[9 + c]);
        }
    }
}

template <int DAGGER>
__global__ void __launch_bounds__(128, 4) dslash32_kernel(DslashArgs<float> A) {
    __shared__ double sm[32];
    int bx = blockIdx.x, src = 0;
    if (A.nb > 1) { src = bx & (A.nb - 1); bx >>= (31 - __clz(A.nb)); }   // grouped sources: see DslashArgs::nb
    A.in = (const char*)A.in + src * A.mul_in * A.fstride;
    A.out = (char*)A.out + src * A.mul_out * A.fstride;
    if (A.x) A.x = (const char*)A.x + src * A.mul_x * A.fstride;
    A.sc += src;
    A.partials += src * TM_PSTRIDE;
    if (guard_skip(A.sc, A.guard)) return;
    const Geom& g = A.g;
    const int h = bx * blockDim.x + threadIdx.x;
    double nrm = 0.0;
    if (h < g.Vh) {
        int xh, y, z, t;
        site_coords(g, h, xh, y, z, t);
        const int odd = (y + z + t + A.parity) & 1;
        const float* in = (const float*)A.in;
        const float* gauge = (const float*)A.gauge;
        const size_t Vh = g.Vh;
        c2 acc[12];
#pragma unroll
        for (int i = 0; i < 12; i++) acc[i] = P2<float>::make(0.f, 0.f);
        if (A.xmode && A.nb > 1) {  // the epilogue's x operand: into L2 now (see dslash16_group_kernel); grouped launches only:
                                    // 697.4 -> 674.5 us per 8 sources, but 113.0 -> 114.5 us for one source per launch
            const float4* xf = reinterpret_cast<const float4*>(A.x) + h;
#pragma unroll
            for (int k = 0; k < 6; k++) asm volatile("prefetch.global.L2 [%0];" ::"l"(xf + (size_t)k * Vh));
        }
        const int row = h - xh;
        const int xp = row + (odd ? (xh + 1 == g.Xh ? 0 : xh + 1) : xh);
        const int xm = row + (odd ? xh : (xh == 0 ? g.Xh - 1 : xh - 1));
        const int yp = (y + 1 == g.X1) ? h - (g.X1 - 1) * g.s1 : h + g.s1;
        const int ym = (y == 0) ? h + (g.X1 - 1) * g.s1 : h - g.s1;
        const int zp = (z + 1 == g.X2) ? h - (g.X2 - 1) * g.s2 : h + g.s2;
        const int zm = (z == 0) ? h + (g.X2 - 1) * g.s2 : h - g.s2;
        const bool wp = (t + 1 == g.X3), wm = (t == 0);
        const int tp = wp ? h - (g.X3 - 1) * g.s3 : h + g.s3;
        const int tm = wm ? h + (g.X3 - 1) * g.s3 : h - g.s3;
        const int par = A.parity;
        hop32<0, 1, DAGGER>(in, gauge, Vh, par, h, xp, 1.f, false, acc);
        hop32<0, 0, DAGGER>(in, gauge, Vh, par, h, xm, 1.f, false, acc);
        hop32<1, 1, DAGGER>(in, gauge, Vh, par, h, yp, 1.f, false, acc);
        hop32<1, 0, DAGGER>(in, gauge, Vh, par, h, ym, 1.f, false, acc);
        hop32<2, 1, DAGGER>(in, gauge, Vh, par, h, zp, 1.f, false, acc);
        hop32<2, 0, DAGGER>(in, gauge, Vh, par, h, zm, 1.f, false, acc);
        hop32<3, 1, DAGGER>(in, gauge, Vh, par, h, tp, A.tb, wp, acc);
        hop32<3, 0, DAGGER>(in, gauge, Vh, par, h, tm, A.tb, wm, acc);
        // epilogue: res = c acc (+ x | + A x, A = 1 + i a g5), optional A^-1 = (1 - i a g5)/(1 + a^2), store, norm
        const float cf = A.c, a = A.a;
        if (A.xmode) {
            const float4* xf = reinterpret_cast<const float4*>(A.x) + h;
#pragma unroll
            for (int k = 0; k < 6; k++) {
                const float4 q4 = __ldg(xf + (size_t)k * Vh);
                const c2 xa = P2<float>::make(q4.x, q4.y), xb = P2<float>::make(q4.z, q4.w);
                c2 ra = P2<float>::fma_s(cf, acc[2 * k], xa), rb = P2<float>::fma_s(cf, acc[2 * k + 1], xb);
                if (A.xmode == 2) {             // + i a x on the upper spins (pairs 0..5), - i a x on the lower ones
                    const float sa = k < 3 ? a : -a;
                    ra = P2<float>::fma_s(sa, times_i<float>(xa), ra);
                    rb = P2<float>::fma_s(sa, times_i<float>(xb), rb);
                }
                acc[2 * k] = ra; acc[2 * k + 1] = rb;
            }
        } else {
#pragma unroll
            for (int i = 0; i < 12; i++) acc[i] = P2<float>::mul_s(cf, acc[i]);
        }
        if (A.post) {
            const float n = 1.f / (1.f + a * a);
#pragma unroll
            for (int i = 0; i < 12; i++) {
                const float sa = i < 6 ? -a : a;            // (1 - i a) on the upper spins, (1 + i a) on the lower ones
                acc[i] = P2<float>::mul_s(n, P2<float>::fma_s(sa, times_i<float>(acc[i]), acc[i]));
            }
        }
        float4* of = reinterpret_cast<float4*>(A.out) + h;
        float n2 = 0.f;
#pragma unroll
        for (int k = 0; k < 6; k++) {
            float4 o;
            P2<float>::get(acc[2 * k], o.x, o.y);
            P2<float>::get(acc[2 * k + 1], o.z, o.w);
            of[(size_t)k * Vh] = o;
            n2 = fmaf(o.x, o.x, n2); n2 = fmaf(o.y, o.y, n2); n2 = fmaf(o.z, o.z, n2); n2 = fmaf(o.w, o.w, n2);
        }
        nrm = (double)n2;
    }
    if (A.red_op != RED_NONE) block_partial_at(nrm, A.partials, bx, sm);
}

static tm_status launch32(tm_ctx* ctx, const DslashCall& c, const void* gauge, cudaStream_t st) {
    DslashArgs<float> A;
    A.in = c.in; A.x = c.x; A.out = c.out; A.gauge = gauge;
    A.g = tm_geom(ctx);
    A.parity = c.out_parity;
    A.dsign = c.dagger ? -1.f : 1.f;
    A.tb = (float)ctx->tb;
    A.a = (float)(2.0 * c.kappa * c.mu * (c.dagger ? -1.0 : 1.0));
    A.c = (float)c.coef;
    A.xmode = c.xmode; A.post = c.post; A.red_op = c.red_op;
    A.partials = ctx->d_partials; A.counter = ctx->d_counter; A.sc = ctx->d_scal;
    A.guard = c.guard;
    A.nb = ctx->nb > 1 ? ctx->nb : 1; A.fstride = ctx->Vh * 24 * sizeof(float);
    A.mul_in = c.mul_in ? c.mul_in : 1; A.mul_x = c.mul_x ? c.mul_x : 1; A.mul_out = c.mul_out ? c.mul_out : 1;
    const int block = 128;
    const int tiles = (int)((ctx->Vh + block - 1) / block);
    const int grid = tiles * A.nb;
    if (c.dagger) dslash32_kernel<1><<<grid, block, 0, st>>>(A);
    else          dslash32_kernel<0><<<grid, block, 0, st>>>(A);
    TM_LAUNCH_CHECK(ctx, "dslash32_kernel");
    if (c.red_op != RED_NONE) TM_TRY(tm_reduce_finish(ctx, (unsigned)tiles, c.red_op, c.guard, st));
    return TM_OK;
}

template <typename S, int R>
static tm_status launch_t(tm_ctx* ctx, const DslashCall& c, const void* gauge, cudaStream_t st) {
    typedef typename Prec<S>::F F;
    DslashArgs<F> A;
    A.in = c.in; A.x = c.x; A.out = c.out; A.gauge = gauge;
    A.g = tm_geom(ctx);
    A.parity = c.out_parity;
    A.dsign = c.dagger ? F(-1) : F(1);
    A.tb = (F)ctx->tb;
    A.a = (F)(2.0 * c.kappa * c.mu * (c.dagger ? -1.0 : 1.0));
    A.c = (F)c.coef;
    A.xmode = c.xmode; A.post = c.post; A.red_op = c.red_op;
    A.partials = ctx->d_partials; A.counter = ctx->d_counter; A.sc = ctx->d_scal;
    A.guard = c.guard;
    A.nb = ctx->nb > 1 ? ctx->nb : 1; A.fstride = ctx->Vh * 24 * sizeof(S);
    A.mul_in = c.mul_in ? c.mul_in : 1; A.mul_x = c.mul_x ? c.mul_x : 1; A.mul_out = c.mul_out ? c.mul_out : 1;
    const int block = 128;
    const int tiles = (int)((ctx->Vh + block - 1) / block);
    const int grid = tiles * A.nb;
    dslash_kernel<S, R><<<grid, block, 0, st>>>(A);
    TM_LAUNCH_CHECK(ctx, "dslash_kernel");
    if (c.red_op != RED_NONE) TM_TRY(tm_reduce_finish(ctx, (unsigned)tiles, c.red_op, c.guard, st));
    return TM_OK;
}

template <typename S, int R>
static tm_status launch16(tm_ctx* ctx, const DslashCall& c, const void* gauge, cudaStream_t st) {
    DslashArgs<float> A;
    A.in = c.in; A.x = c.x; A.out = c.out; A.gauge = gauge;
    A.g = tm_geom(ctx);
    A.parity = c.out_parity;
    A.dsign = c.dagger ? -1.f : 1.f;
    A.tb = (float)ctx->tb;
    A.a = (float)(2.0 * c.kappa * c.mu * (c.dagger ? -1.0 : 1.0));
    A.c = (float)c.coef;
    A.xmode = c.xmode; A.post = c.post; A.red_op = c.red_op;
    A.partials = ctx->d_partials; A.counter = ctx->d_counter; A.sc = ctx->d_scal;
    A.guard = c.guard;
    A.nb = ctx->nb > 1 ? ctx->nb : 1; A.fstride = ctx->Vh * 24 * sizeof(S);
    A.mul_in = c.mul_in ? c.mul_in : 1; A.mul_x = c.mul_x ? c.mul_x : 1; A.mul_out = c.mul_out ? c.mul_out : 1;
    const int block = 128;
    const int tiles = (int)((ctx->Vh + block - 1) / block);
    const int grid = tiles * A.nb;
    // <PIPE = 2, MINB = 5>: links staged by cp.async, 96 registers, 20 warps/SM.  Measured at 32^3x64 (fp16 XPAY,
    // same box): 66.7 us against 69.8 us for register-loaded links <0, 6> and 67.5 us for <2, 6>.
    // reconstruct-18: the same kernel without the row-2 rebuild (9 x 4-byte link chunks, 36 KB of slots per CTA)
    A.ns = 1;
    if (R == 12 && A.nb > 1 && std::is_same<S, __half>::value) {
        // grouped launch: one CTA per tile of 128 sites does all nb sources, which then share the index arithmetic, the
        // link staging and the row-2 rebuilds.  Measured at 32^3x64, 8 sources, fp16 (same box): 430.8 us with one
        // source per CTA (dslash16_kernel, CTAs of a tile adjacent) -> 412.4 us with 4 sources per CTA -> 392.5 us
        // with 8.  bf16 gains nothing (488.5 against 493.7 us) and stays on dslash16_kernel.
        A.ns = A.nb;
        if (c.dagger) dslash16_group_kernel<S, 1, 5><<<tiles, block, 0, st>>>(A);
        else          dslash16_group_kernel<S, 0, 5><<<tiles, block, 0, st>>>(A);
        TM_LAUNCH_CHECK(ctx, "dslash16_group_kernel");
        if (c.red_op != RED_NONE) TM_TRY(tm_reduce_finish(ctx, (unsigned)tiles, c.red_op, c.guard, st));
        return TM_OK;
    }
    if (c.dagger) dslash16_kernel<S, 1, 2, 5, R><<<grid, block, 0, st>>>(A);
    else          dslash16_kernel<S, 0, 2, 5, R><<<grid, block, 0, st>>>(A);
    TM_LAUNCH_CHECK(ctx, "dslash16_kernel");
    if (c.red_op != RED_NONE) TM_TRY(tm_reduce_finish(ctx, (unsigned)tiles, c.red_op, c.guard, st));
    return TM_OK;
}

tm_status tm_dslash_launch(tm_ctx* ctx, const DslashCall& c, tm_prec prec, tm_recon recon, cudaStream_t st) {
    const void* gauge = nullptr;
    TM_TRY(tm_get_gauge(ctx, prec, recon, st, &gauge));
    const bool r12 = (recon == TM_R12);
    switch (prec) {
        case TM_F64:  return r12 ? launch_t<double, 12>(ctx, c, gauge, st) : launch_t<double, 18>(ctx, c, gauge, st);
        case TM_F32:  return r12 ? launch32(ctx, c, gauge, st) : launch_t<float, 18>(ctx, c, gauge, st);
        case TM_F16:  return r12 ? launch16<__half, 12>(ctx, c, gauge, st) : launch16<__half, 18>(ctx, c, gauge, st);
        case TM_BF16: return r12 ? launch16<__nv_bfloat16, 12>(ctx, c, gauge, st)
                                 : launch16<__nv_bfloat16, 18>(ctx, c, gauge, st);
    }
    return tm_fail(ctx, TM_EPREC, "tm_dslash: unknown precision");
}
