// qw_coin.cuh — the per-site coin arithmetic phi = C psi (eq. 1; the inner sum of
// PAPER.md:101 eq. 10), shared by EVERY step kernel of the library so that all schedules
// (generic, fused, temporally blocked, resident) execute the same instruction sequence per site
// and therefore produce bit-identical states.  Every operation is an explicit round-to-nearest
// intrinsic: the compiler may neither contract nor re-associate them.
#pragma once

#include "qw_internal.cuh"

namespace qw {

__device__ __forceinline__ double fma_rn(double a, double b, double c) { return __fma_rn(a, b, c); }
__device__ __forceinline__ float  fma_rn(float a, float b, float c)    { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float  mul_rn(float a, float b)   { return __fmul_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ float  add_rn(float a, float b)   { return __fadd_rn(a, b); }
__device__ __forceinline__ double sub_rn(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ float  sub_rn(float a, float b)   { return __fsub_rn(a, b); }

template <typename R> struct cplx { R re, im; };

template <typename R> __device__ __forceinline__ cplx<R> cx_load(const typename Cx<R>::T *p) {
    typename Cx<R>::T v = *p;
    return cplx<R>{v.x, v.y};
}
template <typename R> __device__ __forceinline__ void cx_store(typename Cx<R>::T *p, cplx<R> z) {
    typename Cx<R>::T v; v.x = z.re; v.y = z.im;
    *p = v;
}

// c * z
template <typename R> __device__ __forceinline__ cplx<R> cx_mul(R cre, R cim, cplx<R> z) {
    cplx<R> r;
    r.re = fma_rn(-cim, z.im, mul_rn(cre, z.re));
    r.im = fma_rn(cim, z.re, mul_rn(cre, z.im));
    return r;
}
// acc + c * z
template <typename R> __device__ __forceinline__ cplx<R> cx_fma(R cre, R cim, cplx<R> z, cplx<R> acc) {
    acc.re = fma_rn(cre, z.re, acc.re);
    acc.re = fma_rn(-cim, z.im, acc.re);
    acc.im = fma_rn(cre, z.im, acc.im);
    acc.im = fma_rn(cim, z.re, acc.im);
    return acc;
}
// ---- complex64 on the packed FP32x2 pipe of sm_100 (FADD2 / FMUL2 / FFMA2: one instruction for re and im) ----------
// IEEE round-to-nearest per component, no flush-to-zero: bit for bit the scalar result, half the issue slots.
#ifndef QW_F32X2
#define QW_F32X2 1
#endif
__device__ __forceinline__ unsigned long long f2_pack(float lo, float hi) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ cplx<float> f2_unpack(unsigned long long v) {
    cplx<float> z;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(z.re), "=f"(z.im) : "l"(v));
    return z;
}
__device__ __forceinline__ cplx<float> f2_add(cplx<float> a, cplx<float> b) {
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_pack(a.re, a.im)), "l"(f2_pack(b.re, b.im)));
    return f2_unpack(r);
}
__device__ __forceinline__ cplx<float> f2_sub(cplx<float> a, cplx<float> b) {
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_pack(a.re, a.im)), "l"(f2_pack(b.re, b.im)));
    return f2_unpack(r);
}
__device__ __forceinline__ cplx<float> f2_mul(float sre, float sim, cplx<float> a) {        // (sre*a.re, sim*a.im)
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_pack(sre, sim)), "l"(f2_pack(a.re, a.im)));
    return f2_unpack(r);
}
__device__ __forceinline__ cplx<float> f2_fma(float sre, float sim, cplx<float> a, cplx<float> b) {   // (sre*a.re + b.re, sim*a.im + b.im)
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(f2_pack(sre, sim)), "l"(f2_pack(a.re, a.im)), "l"(f2_pack(b.re, b.im)));
    return f2_unpack(r);
}

template <typename R> __device__ __forceinline__ cplx<R> cx_add(cplx<R> a, cplx<R> b) {
    if constexpr (QW_F32X2 && sizeof(R) == 4) return f2_add(a, b);
    else return cplx<R>{add_rn(a.re, b.re), add_rn(a.im, b.im)};
}
template <typename R> __device__ __forceinline__ cplx<R> cx_sub(cplx<R> a, cplx<R> b) {
    if constexpr (QW_F32X2 && sizeof(R) == 4) return f2_sub(a, b);
    else return cplx<R>{sub_rn(a.re, b.re), sub_rn(a.im, b.im)};
}
template <typename R> __device__ __forceinline__ cplx<R> cx_scale(R s, cplx<R> a) {
    if constexpr (QW_F32X2 && sizeof(R) == 4) return f2_mul(s, s, a);
    else return cplx<R>{mul_rn(s, a.re), mul_rn(s, a.im)};
}
// s * a + b,  s * a - b  with a real scale s
template <typename R> __device__ __forceinline__ cplx<R> cx_fma_r(R s, cplx<R> a, cplx<R> b) {
    if constexpr (QW_F32X2 && sizeof(R) == 4) return f2_fma(s, s, a, b);
    else return cplx<R>{fma_rn(s, a.re, b.re), fma_rn(s, a.im, b.im)};
}
template <typename R> __device__ __forceinline__ cplx<R> cx_fms_r(R s, cplx<R> a, cplx<R> b) {
    if constexpr (QW_F32X2 && sizeof(R) == 4) return f2_fma(s, s, a, cplx<R>{-b.re, -b.im});
    else return cplx<R>{fma_rn(s, a.re, -b.re), fma_rn(s, a.im, -b.im)};
}
// i * a,  -i * a   (exact)
template <typename R> __device__ __forceinline__ cplx<R> cx_muli(cplx<R> a)  { return cplx<R>{-a.im, a.re}; }
template <typename R> __device__ __forceinline__ cplx<R> cx_mulni(cplx<R> a) { return cplx<R>{a.im, -a.re}; }

// phi = C psi in place.  C: row-major CD x CD complex, interleaved (re, im), rows = output component.
// KIND selects an algebraically equal, cheaper evaluation for the named coins of PAPER.md:82
// (Hadamard, Grover, Fourier) — the host classifies the matrix (qw_api.cu: classify_coin) and only
// picks a special kind when the matrix entries match that pattern exactly.
template <typename R, int CD, int KIND>
__device__ __forceinline__ void apply_coin(const R *__restrict__ C, cplx<R> (&v)[CD]) {
    if constexpr (KIND == COIN_HADAMARD && CD == 2) {
        // s*[[1,1],[1,-1]] as t = s*L; phi_R = s*R + t; phi_L = s*R - t: 2 mul + 4 fma per site
        const R s = C[0];
        const cplx<R> t = cx_scale(s, v[1]), r = v[0];
        v[0] = cx_fma_r(s, r, t);
        v[1] = cx_fms_r(s, r, t);
    } else if constexpr (KIND == COIN_GROVER4 && CD == 4) {
        // off-diagonal g, diagonal d (Grover: g = 1/2, d = -1/2): phi_a = g*sum + (d-g)*psi_a
        const R g = C[2], dg = sub_rn(C[0], C[2]);
        cplx<R> sum = cx_add(cx_add(v[0], v[1]), cx_add(v[2], v[3]));
        cplx<R> gs = cx_scale(g, sum);
#pragma unroll
        for (int a = 0; a < 4; ++a) v[a] = cx_fma_r(dg, v[a], gs);
    } else if constexpr (KIND == COIN_HXH4 && CD == 4) {
        // h * (H (x) H) with c = 2j+k.  The scale rides on the first butterfly (over k) as FMAs:
        // h*(x + y) = fma(h, x, h*y), then the butterfly over j: 2 mul + 4 fma + 4 add per real component.
        // For h = 1/2 (the unitary case) the scaling is exact, i.e. this equals h * ((x + y) + (z + w)) bit for bit.
        const R h = C[0];
        const cplx<R> t1 = cx_scale(h, v[1]), t3 = cx_scale(h, v[3]);
        const cplx<R> a0 = cx_fma_r(h, v[0], t1), a1 = cx_fms_r(h, v[0], t1);
        const cplx<R> a2 = cx_fma_r(h, v[2], t3), a3 = cx_fms_r(h, v[2], t3);
        v[0] = cx_add(a0, a2);
        v[1] = cx_add(a1, a3);
        v[2] = cx_sub(a0, a2);
        v[3] = cx_sub(a1, a3);
    } else if constexpr (KIND == COIN_DFT4 && CD == 4) {
        // h * i^(ab): radix-2 decimation e = h*(v0 +- v2), o = h*(v1 +- v3) with the scale folded into FMAs
        const R h = C[0];
        const cplx<R> t2 = cx_scale(h, v[2]), t3 = cx_scale(h, v[3]);
        const cplx<R> e0 = cx_fma_r(h, v[0], t2), e1 = cx_fms_r(h, v[0], t2);
        const cplx<R> o0 = cx_fma_r(h, v[1], t3), o1 = cx_muli(cx_fms_r(h, v[1], t3));
        v[0] = cx_add(e0, o0);
        v[1] = cx_add(e1, o1);
        v[2] = cx_sub(e0, o0);
        v[3] = cx_sub(e1, o1);
    } else {
        cplx<R> out[CD];
#pragma unroll
        for (int a = 0; a < CD; ++a) {
            cplx<R> acc = cx_mul(C[2 * (a * CD) + 0], C[2 * (a * CD) + 1], v[0]);
#pragma unroll
            for (int b = 1; b < CD; ++b)
                acc = cx_fma(C[2 * (a * CD + b) + 0], C[2 * (a * CD + b) + 1], v[b], acc);
            out[a] = acc;
        }
#pragma unroll
        for (int a = 0; a < CD; ++a) v[a] = out[a];
    }
}

// The named 4x4 coins WITHOUT their overall scale (temporally blocked kernels defer it): the host only classifies a
// matrix as Grover / H(x)H / DFT when that scale (g resp. h) is a power of two, so that multiplying by it commutes
// with every rounding: K bare steps followed by one multiplication by scale^K give bit for bit the state of K
// scaled steps (no overflow: the bare values grow by at most 4^K; underflow to denormals aside).
//   Grover-like  g*sum + (d-g)*psi_a  = g * (sum + r*psi_a),  r = (d-g)/g  (= -2 for the Grover coin)
//   H(x)H, DFT   the radix-2 butterflies of apply_coin with h = 1
template <typename R, int KIND>
__device__ __forceinline__ void apply_coin_bare(R r, cplx<R> (&v)[4]) {
    static_assert(KIND == COIN_GROVER4 || KIND == COIN_HXH4 || KIND == COIN_DFT4, "no bare form for this coin");
    if constexpr (KIND == COIN_GROVER4) {
        const cplx<R> sum = cx_add(cx_add(v[0], v[1]), cx_add(v[2], v[3]));
#pragma unroll
        for (int a = 0; a < 4; ++a) v[a] = cx_fma_r(r, v[a], sum);
    } else if constexpr (KIND == COIN_HXH4) {
        const cplx<R> a0 = cx_add(v[0], v[1]), a1 = cx_sub(v[0], v[1]);
        const cplx<R> a2 = cx_add(v[2], v[3]), a3 = cx_sub(v[2], v[3]);
        v[0] = cx_add(a0, a2);
        v[1] = cx_add(a1, a3);
        v[2] = cx_sub(a0, a2);
        v[3] = cx_sub(a1, a3);
    } else {
        const cplx<R> e0 = cx_add(v[0], v[2]), e1 = cx_sub(v[0], v[2]);
        const cplx<R> o0 = cx_add(v[1], v[3]), o1 = cx_muli(cx_sub(v[1], v[3]));
        v[0] = cx_add(e0, o0);
        v[1] = cx_add(e1, o1);
        v[2] = cx_sub(e0, o0);
        v[3] = cx_sub(e1, o1);
    }
}

// psi = C^dagger phi in place (inverse step; general evaluation only).
template <typename R, int CD>
__device__ __forceinline__ void apply_coin_dagger(const R *__restrict__ C, cplx<R> (&v)[CD]) {
    cplx<R> out[CD];
#pragma unroll
    for (int b = 0; b < CD; ++b) {
        cplx<R> acc = cx_mul(C[2 * (0 * CD + b) + 0], -C[2 * (0 * CD + b) + 1], v[0]);
#pragma unroll
        for (int a = 1; a < CD; ++a)
            acc = cx_fma(C[2 * (a * CD + b) + 0], -C[2 * (a * CD + b) + 1], v[a], acc);
        out[b] = acc;
    }
#pragma unroll
    for (int b = 0; b < CD; ++b) v[b] = out[b];
}

// Direction of coin component `a`: (dm, dn).  1D uses dn only.
template <int DIM>
__device__ __forceinline__ void coin_direction(int lattice, int a, int &dm, int &dn) {
    if constexpr (DIM == 1) {
        dm = 0; dn = (a == 0) ? +1 : -1;                    // R: x+1, L: x-1
    } else {
        if (lattice == QW_NATURAL) {                        // PAPER.md:88 eq. 8, c = 2j+k
            dm = (a == 1) ? +1 : (a == 2 ? -1 : 0);
            dn = (a == 0) ? +1 : (a == 3 ? -1 : 0);
        } else {                                            // PAPER.md:106 Fig. 1c: (m+(-1)^j, n+(-1)^k)
            dm = (a & 2) ? -1 : +1;
            dn = (a & 1) ? -1 : +1;
        }
    }
}

}  // namespace qw
