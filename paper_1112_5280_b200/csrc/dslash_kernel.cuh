// dslash_kernel.cuh -- the Wilson hopping kernel (steps K1-K6 of SURVEY.md sec. 8(a)).
//
//   (H psi)(x) = sum_mu [ (1 - gamma_mu) U_mu(x) psi(x+mu^) + (1 + gamma_mu) U_mu(x-mu^)^+ psi(x-mu^) ]
//
// "the non-diagonal part of the Dirac matrix ('dslash')", even-odd form
// (PAPER.md:61, :87).  One thread per output site.  Chiral gamma basis:
// gamma_mu = [[0, A_mu], [A_mu^+, 0]], A_x,y,z = -i sigma_1,2,3, A_t = -1, so (1 -+ gamma_mu) psi
// is fixed by a two-component half spinor h (K3), the SU(3) multiply acts on h only (K4), and
// the lower two spin components are rebuilt from chi = U h with signs / factors of i (K5).
#pragma once
#include "fields.cuh"
#include "geometry.cuh"

namespace lqcd {

__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }

// unit coefficients: +1, -1, +i, -i
enum Coef { C_P1 = 0, C_M1 = 1, C_PI = 2, C_MI = 3 };
__host__ __device__ constexpr int coef_neg(int c) { return c ^ 1; }
template <int S> __host__ __device__ constexpr int coef_sgn(int c) { return S > 0 ? c : coef_neg(c); }

// d += c * s for a unit coefficient c
template <int C, typename R>
__device__ __forceinline__ void cadd(R& dr, R& di, R sr, R si) {
    if (C == C_P1) { dr += sr; di += si; }
    else if (C == C_M1) { dr -= sr; di -= si; }
    else if (C == C_PI) { dr -= si; di += sr; }
    else { dr += si; di -= sr; }
}

// d += f * c * s for a unit coefficient c and a real factor f
template <int C, typename R>
__device__ __forceinline__ void cfma(R& dr, R& di, R f, R sr, R si) {
    if (C == C_P1) { dr = fma_(f, sr, dr); di = fma_(f, si, di); }
    else if (C == C_M1) { dr = fma_(-f, sr, dr); di = fma_(-f, si, di); }
    else if (C == C_PI) { dr = fma_(-f, si, dr); di = fma_(f, sr, di); }
    else { dr = fma_(f, si, dr); di = fma_(-f, sr, di); }
}

// Projection table: h0 = psi0 + S*ca*psi_ja, h1 = psi1 + S*cb*psi_jb; reconstruction
// r2 = S*c2*chi_k2, r3 = S*c3*chi_k3, with S = +1 for (1 - gamma_mu) (forward hop) and
// S = -1 for (1 + gamma_mu) (backward hop).  Derived from the gamma matrices above.
template <int MU> struct Proj;
template <> struct Proj<0> { static constexpr int ja = 3, ca = C_PI, jb = 2, cb = C_PI, k2 = 1, c2 = C_MI, k3 = 0, c3 = C_MI; };
template <> struct Proj<1> { static constexpr int ja = 3, ca = C_P1, jb = 2, cb = C_M1, k2 = 1, c2 = C_M1, k3 = 0, c3 = C_P1; };
template <> struct Proj<2> { static constexpr int ja = 2, ca = C_PI, jb = 3, cb = C_MI, k2 = 0, c2 = C_MI, k3 = 1, c3 = C_PI; };
template <> struct Proj<3> { static constexpr int ja = 2, ca = C_P1, jb = 3, cb = C_P1, k2 = 0, c2 = C_P1, k3 = 1, c3 = C_P1; };

template <typename R> struct BcPhases { R re[4], im[4]; };

// K3: half spinor h[spin 2][colour 3][reim] = the upper two components of (1 -+ gamma_mu) psi for the forward /
// backward hop (S = +1 / -1), from a gathered neighbour spinor v.
// a + C b for a unit coefficient C on packed complex numbers
template <int C>
__device__ __forceinline__ P2 cadd2(float ar, float ai, float br, float bi) {
    if (C == C_P1) return add2(pk(ar, ai), pk(br, bi));
    if (C == C_M1) return add2(pk(ar, ai), pk(-br, -bi));
    if (C == C_PI) return add2(pk(ar, ai), pk(-bi, br));
    return add2(pk(ar, ai), pk(bi, -br));
}

template <typename R, int MU, int S>
__device__ __forceinline__ void project(const R v[24], R h[12]) {
    using P = Proj<MU>;
    if constexpr (packed_f32<R>) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            unpk(cadd2<coef_sgn<S>(P::ca)>(v[2 * c], v[2 * c + 1], v[6 * P::ja + 2 * c], v[6 * P::ja + 2 * c + 1]), h[2 * c], h[2 * c + 1]);
            unpk(cadd2<coef_sgn<S>(P::cb)>(v[6 + 2 * c], v[6 + 2 * c + 1], v[6 * P::jb + 2 * c], v[6 * P::jb + 2 * c + 1]), h[6 + 2 * c], h[6 + 2 * c + 1]);
        }
        return;
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        R r0 = v[2 * c], i0 = v[2 * c + 1];
        cadd<coef_sgn<S>(P::ca)>(r0, i0, v[6 * P::ja + 2 * c], v[6 * P::ja + 2 * c + 1]);
        R r1 = v[6 + 2 * c], i1 = v[6 + 2 * c + 1];
        cadd<coef_sgn<S>(P::cb)>(r1, i1, v[6 * P::jb + 2 * c], v[6 * P::jb + 2 * c + 1]);
        h[2 * c] = r0; h[2 * c + 1] = i0;
        h[6 + 2 * c] = r1; h[6 + 2 * c + 1] = i1;
    }
}

// K3 on 16-bit storage with Blackwell's mixed-precision adds (add/sub.rn.f32.f16 -> FHADD: an f16 operand taken from
// either half of a register plus an f32 operand, exact fp32 result): the lower spin component is converted (12
// conversions per hop instead of 24) and the upper one enters the add as f16, so the projection costs no rounding and
// no instruction beyond the conversion it replaces.  w: the 3 16-byte words of the site, complex k = 3 spin + colour
// in 32-bit register k (low half re, high half im).
__device__ __forceinline__ float fhadd(unsigned short a, float c) { float r; asm("add.rn.f32.f16 %0, %1, %2;" : "=f"(r) : "h"(a), "f"(c)); return r; }
__device__ __forceinline__ float fhsub(unsigned short a, float c) { float r; asm("sub.rn.f32.f16 %0, %1, %2;" : "=f"(r) : "h"(a), "f"(c)); return r; }

// (re, im) = a + C b for a unit coefficient C; a, b packed half2 (re low, im high)
template <int C>
__device__ __forceinline__ void cmix_h(unsigned a, unsigned b, float& re, float& im) {
    const unsigned short ar = (unsigned short)(a & 0xffffu), ai = (unsigned short)(a >> 16);
    const float2 bf = __half22float2(*reinterpret_cast<const __half2*>(&b));
    if (C == C_P1) { re = fhadd(ar, bf.x); im = fhadd(ai, bf.y); }
    else if (C == C_M1) { re = fhsub(ar, bf.x); im = fhsub(ai, bf.y); }
    else if (C == C_PI) { re = fhsub(ar, bf.y); im = fhadd(ai, bf.x); }
    else { re = fhadd(ar, bf.y); im = fhsub(ai, bf.x); }
}

template <int MU, int S>
__device__ __forceinline__ void project_h(const uint4 w[3], float h[12]) {
    using P = Proj<MU>;
    const unsigned* k = reinterpret_cast<const unsigned*>(w);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        cmix_h<coef_sgn<S>(P::ca)>(k[c], k[3 * P::ja + c], h[2 * c], h[2 * c + 1]);
        cmix_h<coef_sgn<S>(P::cb)>(k[3 + c], k[3 * P::jb + c], h[6 + 2 * c], h[6 + 2 * c + 1]);
    }
}

// K3b: psi(x + L mu^) = bc psi(x): forward crossing multiplies by bc_mu = br + i bi, backward by its conjugate (the
// caller passes -bi).  Real (+-1) phases cost nothing: the sign rides on the accumulation factor f of K5, and so does the
// site norm of 16-bit storage (the neighbour spinor is scale * v; the hop is linear).  Returns f.
template <typename R, bool CBC>
__device__ __forceinline__ R boundary_phase(R h[12], R scale, bool cross, R br, R bi) {
    if (CBC) {
        if (cross) {
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                const R a = h[2 * k], b = h[2 * k + 1];
                h[2 * k] = a * br - b * bi;
                h[2 * k + 1] = a * bi + b * br;
            }
        }
        return scale;
    }
    return cross ? br * scale : scale;
}

// K4: chi = U h (forward) or U^+ h (backward), both spin components; explicit FMA chains
template <typename R, bool FWD>
__device__ __forceinline__ void su3_multiply(const R h[12], const R u[18], R chi[12]) {
    if constexpr (packed_f32<R>) {
        // (re, im) as one pair: P = sum_b ur (hr, hi), Q = sum_b ui (hi, hr); forward chi = (P.x - Q.x, P.y + Q.y),
        // backward (conjugated link) chi = (P.x + Q.x, P.y - Q.y): 2 FFMA2 per complex multiply-add, 1 FADD2 per output
#pragma unroll
        for (int sp = 0; sp < 2; ++sp)
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                P2 pp, qq;
#pragma unroll
                for (int b = 0; b < 3; ++b) {
                    const float hr = h[6 * sp + 2 * b], hi = h[6 * sp + 2 * b + 1];
                    const float ur = FWD ? u[6 * a + 2 * b] : u[6 * b + 2 * a];
                    const float ui = FWD ? u[6 * a + 2 * b + 1] : u[6 * b + 2 * a + 1];
                    pp = b == 0 ? mul2(bc2(ur), pk(hr, hi)) : fma2(bc2(ur), pk(hr, hi), pp);
                    qq = b == 0 ? mul2(bc2(ui), pk(hi, hr)) : fma2(bc2(ui), pk(hi, hr), qq);
                }
                float qx, qy;
                unpk(qq, qx, qy);
                unpk(add2(pp, FWD ? pk(-qx, qy) : pk(qx, -qy)), chi[6 * sp + 2 * a], chi[6 * sp + 2 * a + 1]);
            }
        return;
    }
#pragma unroll
    for (int sp = 0; sp < 2; ++sp)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            R cr, ci;
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                const R hr = h[6 * sp + 2 * b], hi = h[6 * sp + 2 * b + 1];
                // forward: U[a][b];  backward: conj(U[b][a])
                const R ur = FWD ? u[6 * a + 2 * b] : u[6 * b + 2 * a];
                const R ui = FWD ? u[6 * a + 2 * b + 1] : -u[6 * b + 2 * a + 1];
                if (b == 0) {
                    cr = ur * hr;
                    ci = ur * hi;
                } else {
                    cr = fma_(ur, hr, cr);
                    ci = fma_(ur, hi, ci);
                }
                cr = fma_(-ui, hi, cr);
                ci = fma_(ui, hr, ci);
            }
            chi[6 * sp + 2 * a] = cr;
            chi[6 * sp + 2 * a + 1] = ci;
        }
}

// K5: out0 += f chi0, out1 += f chi1, out2 += f S c2 chi_k2, out3 += f S c3 chi_k3
// d += f c s for a unit coefficient c, packed
template <int C>
__device__ __forceinline__ void cfma2(float& dr, float& di, float f, float sr, float si) {
    P2 d = pk(dr, di);
    if (C == C_P1) d = fma2(bc2(f), pk(sr, si), d);
    else if (C == C_M1) d = fma2(bc2(-f), pk(sr, si), d);
    else if (C == C_PI) d = fma2(pk(-f, f), pk(si, sr), d);    // dr += -f si, di += f sr
    else d = fma2(pk(f, -f), pk(si, sr), d);                   // dr += f si, di += -f sr
    unpk(d, dr, di);
}

template <typename R, int MU, int S>
__device__ __forceinline__ void reconstruct_accumulate(R acc[24], const R chi[12], R f) {
    using P = Proj<MU>;
    if constexpr (packed_f32<R>) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            cfma2<C_P1>(acc[2 * c], acc[2 * c + 1], f, chi[2 * c], chi[2 * c + 1]);
            cfma2<C_P1>(acc[6 + 2 * c], acc[6 + 2 * c + 1], f, chi[6 + 2 * c], chi[6 + 2 * c + 1]);
            cfma2<coef_sgn<S>(P::c2)>(acc[12 + 2 * c], acc[12 + 2 * c + 1], f, chi[6 * P::k2 + 2 * c], chi[6 * P::k2 + 2 * c + 1]);
            cfma2<coef_sgn<S>(P::c3)>(acc[18 + 2 * c], acc[18 + 2 * c + 1], f, chi[6 * P::k3 + 2 * c], chi[6 * P::k3 + 2 * c + 1]);
        }
        return;
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        acc[2 * c] = fma_(f, chi[2 * c], acc[2 * c]);
        acc[2 * c + 1] = fma_(f, chi[2 * c + 1], acc[2 * c + 1]);
        acc[6 + 2 * c] = fma_(f, chi[6 + 2 * c], acc[6 + 2 * c]);
        acc[6 + 2 * c + 1] = fma_(f, chi[6 + 2 * c + 1], acc[6 + 2 * c + 1]);
        cfma<coef_sgn<S>(P::c2)>(acc[12 + 2 * c], acc[12 + 2 * c + 1], f, chi[6 * P::k2 + 2 * c], chi[6 * P::k2 + 2 * c + 1]);
        cfma<coef_sgn<S>(P::c3)>(acc[18 + 2 * c], acc[18 + 2 * c + 1], f, chi[6 * P::k3 + 2 * c], chi[6 * P::k3 + 2 * c + 1]);
    }
}

// The rest of the arithmetic of one hop on the projected half spinor h and the link u:
// boundary phase (K3b), colour multiply (K4), reconstruct + accumulate (K5).
template <typename R, bool CBC, int MU, bool FWD>
__device__ __forceinline__ void hop_rest(R acc[24], R h[12], R scale, const R u[18], bool cross, const BcPhases<R>& bc) {
    const R f = boundary_phase<R, CBC>(h, scale, cross, bc.re[MU], FWD ? bc.im[MU] : -bc.im[MU]);
    R chi[12];
    su3_multiply<R, FWD>(h, u, chi);
    reconstruct_accumulate<R, MU, FWD ? +1 : -1>(acc, chi, f);
}

// 16-bit storage, arithmetic on the stored operands (LQCD_F16_MIXED = 2).  Blackwell multiplies two f16 operands into an
// f32 accumulator (fma.rn.f32.f16 -> FHFMA; either half of a 32-bit register, with negation, is an operand): the
// product of two 11-bit significands is exact in f32, so the SU(3) multiply needs no conversion of the links or of the
// half spinor at all -- provided the half spinor is an f16 quantity.  So: K3 projects in packed half arithmetic
// (h = v_a + c v_b rounded once to f16; 6 instructions per hop instead of 24 conversions + 12 adds), K2 rebuilds the
// third link row in f32 from exact f16 products and rounds it to f16 like the two stored rows, K4 runs on FHFMA with
// f32 accumulation, K5 and the epilogue stay f32.  Two roundings to an 11-bit significand are added per hop (the
// projected half spinor and the rebuilt row); DESIGN.md "16-bit storage" derives what they cost: ~1.5e-4 in rel-L2.
__device__ __forceinline__ float fhfma(unsigned short a, unsigned short b, float c) {
    float r; asm("fma.rn.f32.f16 %0, %1, %2, %3;" : "=f"(r) : "h"(a), "h"(b), "f"(c)); return r;
}
__device__ __forceinline__ float fhfnma(unsigned short a, unsigned short b, float c) {   // c - a b
    float r; asm("{ .reg .f16 t; neg.f16 t, %1; fma.rn.f32.f16 %0, t, %2, %3; }" : "=f"(r) : "h"(a), "h"(b), "f"(c)); return r;
}
__device__ __forceinline__ unsigned short lo16(unsigned x) { return (unsigned short)(x & 0xffffu); }
__device__ __forceinline__ unsigned short hi16(unsigned x) { return (unsigned short)(x >> 16); }

// a + C b for a unit coefficient C on packed f16 complex numbers (re low, im high), rounded to f16
template <int C>
__device__ __forceinline__ unsigned cmix_hh(unsigned a, unsigned b) {
    const __half2 A = *reinterpret_cast<const __half2*>(&a), B = *reinterpret_cast<const __half2*>(&b);
    __half2 r;
    if (C == C_P1) r = __hadd2(A, B);
    else if (C == C_M1) r = __hsub2(A, B);
    else if (C == C_PI) r = __hfma2(__lowhigh2highlow(B), __floats2half2_rn(-1.f, 1.f), A);   // (ar - bi, ai + br)
    else r = __hfma2(__lowhigh2highlow(B), __floats2half2_rn(1.f, -1.f), A);                 // (ar + bi, ai - br)
    return *reinterpret_cast<const unsigned*>(&r);
}

// K3 on the stored words: hh[3 sp + c] = packed f16 complex, spin component sp of the projected half spinor
template <int MU, int S>
__device__ __forceinline__ void project_hh(const uint4 w[3], unsigned hh[6]) {
    using P = Proj<MU>;
    const unsigned* k = reinterpret_cast<const unsigned*>(w);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        hh[c] = cmix_hh<coef_sgn<S>(P::ca)>(k[c], k[3 * P::ja + c]);
        hh[3 + c] = cmix_hh<coef_sgn<S>(P::cb)>(k[3 + c], k[3 * P::jb + c]);
    }
}

// L1 + K2: the two stored rows as 6 packed f16 complex numbers u[3 row + col], the third row rebuilt as
// conj(row0 x row1) in f32 (exact products) and rounded to f16: u[6 + col]
__device__ __forceinline__ void load_link_hh(const uint2* __restrict__ site_links, int k, unsigned u[9]) {
#pragma unroll
    for (int w = 0; w < 3; ++w) {
        const uint2 x = __ldcs(site_links + (k * 3 + w) * TILE);
        u[2 * w] = x.x;
        u[2 * w + 1] = x.y;
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int a = (c + 1) % 3, b = (c + 2) % 3;
        const unsigned A = u[a], B = u[b], C = u[3 + b], D = u[3 + a];
        float re = fhfma(lo16(A), lo16(C), 0.f);
        re = fhfnma(hi16(A), hi16(C), re);
        re = fhfnma(lo16(B), lo16(D), re);
        re = fhfma(hi16(B), hi16(D), re);
        float im = fhfma(lo16(A), hi16(C), 0.f);
        im = fhfma(hi16(A), lo16(C), im);
        im = fhfnma(lo16(B), hi16(D), im);
        im = fhfnma(hi16(B), lo16(D), im);
        const __half2 r = __floats2half2_rn(re, -im);
        u[6 + c] = *reinterpret_cast<const unsigned*>(&r);
    }
}

// K4 on f16 operands, f32 accumulation: chi = U h (forward) or U^+ h (backward)
template <bool FWD>
__device__ __forceinline__ void su3_multiply_hh(const unsigned hh[6], const unsigned u[9], float chi[12]) {
#pragma unroll
    for (int sp = 0; sp < 2; ++sp)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            float cr = 0.f, ci = 0.f;
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                const unsigned h = hh[3 * sp + b], U = FWD ? u[3 * a + b] : u[3 * b + a];
                if (FWD) {   // (ur + i ui)(hr + i hi)
                    cr = fhfma(lo16(U), lo16(h), cr);
                    cr = fhfnma(hi16(U), hi16(h), cr);
                    ci = fhfma(lo16(U), hi16(h), ci);
                    ci = fhfma(hi16(U), lo16(h), ci);
                } else {     // (ur - i ui)(hr + i hi)
                    cr = fhfma(lo16(U), lo16(h), cr);
                    cr = fhfma(hi16(U), hi16(h), cr);
                    ci = fhfma(lo16(U), hi16(h), ci);
                    ci = fhfnma(hi16(U), lo16(h), ci);
                }
            }
            chi[6 * sp + 2 * a] = cr;
            chi[6 * sp + 2 * a + 1] = ci;
        }
}

// one hop of the 16-bit kernel on stored operands
template <bool CBC, int K>
__device__ __forceinline__ void hop_step_hh(float acc[24], const uint2* __restrict__ site_links, const __half* __restrict__ in, int ntiles,
                                            const int nb[8], unsigned crossmask, const BcPhases<float>& bc) {
    constexpr int MU = K / 2;
    constexpr bool FWD = (K & 1) == 0;
    uint4 w[3];
    float scale;
    load_words_h(in, ntiles, nb[K], w, scale);
    unsigned hh[6], u[9];
    project_hh<MU, FWD ? +1 : -1>(w, hh);
    load_link_hh(site_links, K, u);
    float chi[12];
    su3_multiply_hh<FWD>(hh, u, chi);
    // K3b on chi instead of h (the multiply is linear): psi(x + L mu^) = bc psi(x)
    const bool cross = (crossmask >> K) & 1u;
    const float f = boundary_phase<float, CBC>(chi, scale, cross, bc.re[MU], FWD ? bc.im[MU] : -bc.im[MU]);
    reconstruct_accumulate<float, MU, FWD ? +1 : -1>(acc, chi, f);
}

// 16-bit storage: 2 = arithmetic on the stored f16 operands (above); 1 = exact projection with mixed-precision adds, the
// rest in f32 after conversion; 0 = convert all 24 components and the link first
#ifndef LQCD_F16_MIXED
#define LQCD_F16_MIXED 2
#endif

// Hop K = 2 mu + (backward ? 1 : 0): gather the neighbour spinor and the link stored for this hop
// (U_mu(x) or U_mu(x - mu^), fields.cuh), then the arithmetic.  S = storage type, R = arithmetic type.
template <typename S, int RECON, bool CBC, int K>
__device__ __forceinline__ void hop_step(typename Compute<S>::type acc[24],
                                         const typename LinkStore<S, RECON>::word* __restrict__ site_links,
                                         const S* __restrict__ in, int ntiles, const int nb[8], unsigned crossmask,
                                         const BcPhases<typename Compute<S>::type>& bc) {
    using R = typename Compute<S>::type;
    constexpr int MU = K / 2;
    constexpr bool FWD = (K & 1) == 0;
    if constexpr (sizeof(S) == 2 && LQCD_F16_MIXED == 2) {
        hop_step_hh<CBC, K>(acc, site_links, in, ntiles, nb, crossmask, bc);
        return;
    }
    R h[12], u[18], scale;
    if constexpr (sizeof(S) == 2 && LQCD_F16_MIXED) {
        uint4 w[3];
        load_words_h(in, ntiles, nb[K], w, scale);
        project_h<MU, FWD ? +1 : -1>(w, h);
    } else {
        R v[24];
        load_field<S>(in, ntiles, nb[K], v, scale);
        project<R, MU, FWD ? +1 : -1>(v, h);
    }
    if constexpr (half_links<S, RECON>) load_link_h(site_links, K, u); else load_link<R, RECON>(site_links, K, u);
    hop_rest<R, CBC, MU, FWD>(acc, h, scale, u, (crossmask >> K) & 1u, bc);
}

// Resident 64-thread blocks per SM promised to ptxas (__launch_bounds__ min blocks).  The hint sets the
// register budget (65536 / (64 value)), and ptxas spends whatever budget it is given on hoisting the
// gathers ahead of their use, so it fixes the balance between loads in flight per thread and threads
// per SM.  Values measured on B200 at 32^3x64 (profiles/r01_varsweep_minblocks.txt); overridable for sweeps.
#ifndef LQCD_MINB_F32_R12
#define LQCD_MINB_F32_R12 8
#endif
#ifndef LQCD_MINB_F32_R18
#define LQCD_MINB_F32_R18 6
#endif
#ifndef LQCD_MINB_F64_R12
#define LQCD_MINB_F64_R12 6
#endif
#ifndef LQCD_MINB_F64_R18
#define LQCD_MINB_F64_R18 4
#endif
#ifndef LQCD_MINB_F16_R12
#define LQCD_MINB_F16_R12 10
#endif
#ifndef LQCD_MINB_F32_R8
#define LQCD_MINB_F32_R8 8
#endif
#ifndef LQCD_MINB_F64_R8
#define LQCD_MINB_F64_R8 6
#endif
template <typename R, int RECON> struct MinBlocks;
template <> struct MinBlocks<float, 12>  { static constexpr int value = LQCD_MINB_F32_R12; };
template <> struct MinBlocks<float, 18>  { static constexpr int value = LQCD_MINB_F32_R18; };
template <> struct MinBlocks<double, 12> { static constexpr int value = LQCD_MINB_F64_R12; };
template <> struct MinBlocks<double, 18> { static constexpr int value = LQCD_MINB_F64_R18; };
template <> struct MinBlocks<__half, 12>  { static constexpr int value = LQCD_MINB_F16_R12; };
template <> struct MinBlocks<float, 8>   { static constexpr int value = LQCD_MINB_F32_R8; };
template <> struct MinBlocks<double, 8>  { static constexpr int value = LQCD_MINB_F64_R8; };
#ifndef LQCD_MINB_F32_R12H
#define LQCD_MINB_F32_R12H 8
#endif
template <> struct MinBlocks<float, RECON_12H> { static constexpr int value = LQCD_MINB_F32_R12H; };

// Step K6, the epilogue applied to acc = (H in)(x) before the store (EPI):
//   EPI_STORE    out = acc                                        lqcd_dslash_*
//   EPI_XPAY     out = x + a acc                                  lqcd_apply_M   (a = -kappa or -kappa^2)
//   EPI_G5SCALE  out = (g_re + i g_im gamma_5) acc                lqcd_apply_M_tm, first pass: (1 + i theta g5)^-1 H_oe in
//   EPI_G5XPAY   out = (g_re + i g_im gamma_5) x + a acc          lqcd_apply_M_tm, last pass:  (1 + i theta g5) in - kappa^2 H ...
// With g5_out the stored result is gamma_5 times the above (Q = gamma_5 M, the operator CG works with).
// gamma_5 = diag(1, 1, -1, -1) in the chiral basis, so the twisted-mass site-diagonal term is a complex
// scalar on the upper two spin components and its conjugate on the lower two: it costs no extra memory traffic.
enum { EPI_STORE = 0, EPI_XPAY = 1, EPI_G5SCALE = 2, EPI_G5XPAY = 3 };
template <typename R> struct Epilogue { R a, g_re, g_im; int g5_out; };  // g5_out: finally out <- gamma_5 out

// v <- (g_re + i g_im gamma_5) v
template <typename R>
__device__ __forceinline__ void g5_scale(R v[24], R g_re, R g_im) {
#pragma unroll
    for (int k = 0; k < 12; ++k) {
        const R gi = k < 6 ? g_im : -g_im;
        const R re = v[2 * k], im = v[2 * k + 1];
        v[2 * k] = fma_(-gi, im, g_re * re);
        v[2 * k + 1] = fma_(gi, re, g_re * im);
    }
}

// K6 + L6: the epilogue on acc = (H in)(x), then the store (shared by the gather kernel and the pipelined kernel).
template <typename S, int EPI>
__device__ __forceinline__ void finish_site(typename Compute<S>::type acc[24], S* __restrict__ out, const S* __restrict__ xin,
                                            const Epilogue<typename Compute<S>::type>& epi, int ntiles, int cb, bool live) {
    using R = typename Compute<S>::type;
    constexpr bool XPAY = EPI == EPI_XPAY || EPI == EPI_G5XPAY;
    if constexpr (EPI == EPI_G5SCALE) g5_scale<R>(acc, epi.g_re, epi.g_im);
    if constexpr (XPAY) {
        R x[24], xs;
        load_field<S>(xin, ntiles, cb, x, xs);
        if constexpr (sizeof(S) == 2) {
#pragma unroll
            for (int k = 0; k < 24; ++k) x[k] *= xs;
        }
        if constexpr (EPI == EPI_G5XPAY) g5_scale<R>(x, epi.g_re, epi.g_im);
#pragma unroll
        for (int k = 0; k < 24; ++k) acc[k] = fma_(epi.a, acc[k], x[k]);
    }
    if (epi.g5_out) {
#pragma unroll
        for (int k = 12; k < 24; ++k) acc[k] = -acc[k];
    }
    if (live) store_field<S>(out, ntiles, cb, acc);
}

// Thread -> site maps.  Linear: thread t of block b works on checkerboard site cb_begin + b BLOCK + t (a block is a run of
// consecutive sites: 4 x-rows at 32^3 x 64).  Blocked (whole-lattice launches on lattices whose z planes are multiples of
// 32 sites): the warp tiles form a 3-D grid (ny tiles per z plane) x Z x T, and a block of by bz bt warps takes a compact
// by x bz x bt box of it -- a 4-D sub-volume of the lattice -- so that the neighbour spinors its warps gather are to a
// large part the same tiles and are served by the SM's L1 instead of crossing the L2 -> SM crossbar again (the kernel is
// bound by that crossbar, not by HBM: DESIGN.md section 6).  by = 0: linear.
struct BlockMap { int by, bz, bt, ny, gy, gz; };   // box shape in tiles; tiles per z plane; blocks along y, z

// grid.y = 1: one parity `parity0`; grid.y = 2: both, parity = blockIdx.y, and in/out/xin are
// full fields [even|odd] (in is read at the opposite half).  One thread per output site.
// S = storage type of all fields (float, double, or __half with fp32 arithmetic), R = arithmetic type.
template <typename S, int RECON, int EPI, bool CBC, int BLOCK>
__global__ void __launch_bounds__(BLOCK, MinBlocks<S, RECON>::value * 64 / BLOCK)
dslash_kernel(S* __restrict__ out, const S* __restrict__ gauge, const S* __restrict__ in, const S* __restrict__ xin,
              Epilogue<typename Compute<S>::type> epi, Geom g, int parity0, BcPhases<typename Compute<S>::type> bc,
              int cb_begin, int cb_end, BlockMap map) {
    using R = typename Compute<S>::type;
    constexpr bool XPAY = EPI == EPI_XPAY || EPI == EPI_G5XPAY;
    int p = parity0;
    if (gridDim.y == 2) {
        p = blockIdx.y;
        const size_t half = half_stride<S>(g.ntiles);
        in += (size_t)(1 - p) * half;
        out += (size_t)p * half;
        if (XPAY) xin += (size_t)p * half;
    }
    int cb = cb_begin + blockIdx.x * BLOCK + threadIdx.x;  // [cb_begin, cb_end): all sites, or a range of time slices
    if (map.by) {
        const int w = threadIdx.x >> 5, b = blockIdx.x;
        const int wy = w % map.by, wz = (w / map.by) % map.bz, wt = w / (map.by * map.bz);
        const int gy = b % map.gy, gz = (b / map.gy) % map.gz, gt = b / (map.gy * map.gz);
        const int ty = gy * map.by + wy, tz = gz * map.bz + wz, tt = gt * map.bt + wt;
        if (ty >= map.ny || tz >= g.Z || tt >= g.T) return;   // boxes that stick out of the lattice (warp-uniform)
        cb = (ty + map.ny * (tz + g.Z * tt)) * TILE + (int)(threadIdx.x & 31u);
    }
    if (cb >= cb_end) return;
    const Site s = decode_site(g, cb, p);

    // K1: all eight neighbours and boundary-crossing flags
    int nb[8];
    unsigned crossmask;
    all_neighbours(g, cb, s, nb, crossmask);
    const auto* site_links = reinterpret_cast<const typename LinkStore<S, RECON>::word*>(gauge) +
                             LinkStore<S, RECON>::word0(g.ntiles, p, cb, 0);

    R acc[24];
#pragma unroll
    for (int k = 0; k < 24; ++k) acc[k] = 0;

    hop_step<S, RECON, CBC, 0>(acc, site_links, in, g.ntiles, nb, crossmask, bc);
    hop_step<S, RECON, CBC, 1>(acc, site_links, in, g.ntiles, nb, crossmask, bc);
    hop_step<S, RECON, CBC, 2>(acc, site_links, in, g.ntiles, nb, crossmask, bc);
    hop_step<S, RECON, CBC, 3>(acc, site_links, in, g.ntiles, nb, crossmask, bc);
    hop_step<S, RECON, CBC, 4>(acc, site_links, in, g.ntiles, nb, crossmask, bc);
    hop_step<S, RECON, CBC, 5>(acc, site_links, in, g.ntiles, nb, crossmask, bc);
    hop_step<S, RECON, CBC, 6>(acc, site_links, in, g.ntiles, nb, crossmask, bc);
    hop_step<S, RECON, CBC, 7>(acc, site_links, in, g.ntiles, nb, crossmask, bc);

    finish_site<S, EPI>(acc, out, xin, epi, g.ntiles, cb, true);
}

}  // namespace lqcd
