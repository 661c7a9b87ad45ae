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

// Projection table: h0 = psi0 + S*ca*psi_ja, h1 = psi1 + S*cb*psi_jb; reconstruction
// r2 = S*c2*chi_k2, r3 = S*c3*chi_k3, with S = +1 for (1 - gamma_mu) (forward hop) and
// S = -1 for (1 + gamma_mu) (backward hop).  Derived from the gamma matrices above.
template <int MU> struct Proj;
template <> struct Proj<0> { static constexpr int ja = 3, ca = C_PI, jb = 2, cb = C_PI, k2 = 1, c2 = C_MI, k3 = 0, c3 = C_MI; };
template <> struct Proj<1> { static constexpr int ja = 3, ca = C_P1, jb = 2, cb = C_M1, k2 = 1, c2 = C_M1, k3 = 0, c3 = C_P1; };
template <> struct Proj<2> { static constexpr int ja = 2, ca = C_PI, jb = 3, cb = C_MI, k2 = 0, c2 = C_MI, k3 = 1, c3 = C_PI; };
template <> struct Proj<3> { static constexpr int ja = 2, ca = C_P1, jb = 3, cb = C_P1, k2 = 0, c2 = C_P1, k3 = 1, c3 = C_P1; };

template <typename R> struct BcPhases { R re[4], im[4]; };

// One of the eight hops: gather neighbour spinor, project (K3), boundary phase (K3b),
// colour multiply (K4), reconstruct + accumulate (K5).
template <typename R, int RECON, bool CBC, int MU, bool FWD>
__device__ __forceinline__ void hop(R acc[24], const R* __restrict__ gauge, const R* __restrict__ in,
                                    const Geom& g, int cb, const Site& s, int p, const BcPhases<R>& bc) {
    constexpr int S = FWD ? +1 : -1;
    using P = Proj<MU>;
    bool cross;
    const int nb = neighbour<MU, FWD>(g, cb, s, cross);

    R v[24];
    load_spinor<R>(in, g.Vh, nb, v);
    R u[18];
    // forward link U_mu(x) lives at x (parity p); backward link U_mu(x-mu^) at the neighbour (parity 1-p)
    load_link<R, RECON>(gauge, g.Vh, FWD ? p : 1 - p, MU, FWD ? cb : nb, u);

    // K3: half spinor h[spin 2][colour 3][reim]
    R h[12];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        R r0 = v[2 * c], i0 = v[2 * c + 1];
        cadd<coef_sgn<S>(P::ca)>(r0, i0, v[6 * P::ja + 2 * c], v[6 * P::ja + 2 * c + 1]);
        R r1 = v[6 + 2 * c], i1 = v[6 + 2 * c + 1];
        cadd<coef_sgn<S>(P::cb)>(r1, i1, v[6 * P::jb + 2 * c], v[6 * P::jb + 2 * c + 1]);
        h[2 * c] = r0; h[2 * c + 1] = i0;
        h[6 + 2 * c] = r1; h[6 + 2 * c + 1] = i1;
    }

    // K3b: psi(x + L mu^) = bc psi(x): forward crossing multiplies by bc_mu, backward by conj(bc_mu)
    if (CBC) {
        if (cross) {
            const R br = bc.re[MU], bi = FWD ? bc.im[MU] : -bc.im[MU];
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                const R a = h[2 * k], b = h[2 * k + 1];
                h[2 * k] = a * br - b * bi;
                h[2 * k + 1] = a * bi + b * br;
            }
        }
    } else {
        const R f = cross ? bc.re[MU] : R(1);  // +-1
#pragma unroll
        for (int k = 0; k < 12; ++k) h[k] *= f;
    }

    // K4: chi = U h (forward) or U^+ h (backward), both spin components
    R chi[12];
#pragma unroll
    for (int sp = 0; sp < 2; ++sp)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            R cr = 0, ci = 0;
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                const R hr = h[6 * sp + 2 * b], hi = h[6 * sp + 2 * b + 1];
                if (FWD) {
                    const R ur = u[6 * a + 2 * b], ui = u[6 * a + 2 * b + 1];
                    cr += ur * hr - ui * hi;
                    ci += ur * hi + ui * hr;
                } else {  // conj(U[b][a])
                    const R ur = u[6 * b + 2 * a], ui = u[6 * b + 2 * a + 1];
                    cr += ur * hr + ui * hi;
                    ci += ur * hi - ui * hr;
                }
            }
            chi[6 * sp + 2 * a] = cr;
            chi[6 * sp + 2 * a + 1] = ci;
        }

    // K5: out0 += chi0, out1 += chi1, out2 += S c2 chi_k2, out3 += S c3 chi_k3
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        acc[2 * c] += chi[2 * c];
        acc[2 * c + 1] += chi[2 * c + 1];
        acc[6 + 2 * c] += chi[6 + 2 * c];
        acc[6 + 2 * c + 1] += chi[6 + 2 * c + 1];
        cadd<coef_sgn<S>(P::c2)>(acc[12 + 2 * c], acc[12 + 2 * c + 1], chi[6 * P::k2 + 2 * c], chi[6 * P::k2 + 2 * c + 1]);
        cadd<coef_sgn<S>(P::c3)>(acc[18 + 2 * c], acc[18 + 2 * c + 1], chi[6 * P::k3 + 2 * c], chi[6 * P::k3 + 2 * c + 1]);
    }
}

// out_p(x) = (H in)(x)              (XPAY = false)
// out_p(x) = xin(x) + a (H in)(x)    (XPAY = true; a = -kappa or -kappa^2, step K6)
// grid.y = 1: one parity `parity0`; grid.y = 2: both, parity = blockIdx.y, and in/out/xin are
// full fields [even|odd] (in is read at the opposite half).
template <typename R, int RECON, bool XPAY, bool CBC, int BLOCK>
__global__ void __launch_bounds__(BLOCK)
dslash_kernel(R* __restrict__ out, const R* __restrict__ gauge, const R* __restrict__ in,
              const R* __restrict__ xin, R a, Geom g, int parity0, BcPhases<R> bc) {
    const int cb = blockIdx.x * BLOCK + threadIdx.x;
    if (cb >= g.Vh) return;
    int p = parity0;
    if (gridDim.y == 2) {
        p = blockIdx.y;
        const size_t half = (size_t)24 * g.Vh;
        in += (size_t)(1 - p) * half;
        out += (size_t)p * half;
        if (XPAY) xin += (size_t)p * half;
    }
    const Site s = decode_site(g, cb, p);

    R acc[24];
#pragma unroll
    for (int k = 0; k < 24; ++k) acc[k] = 0;

    hop<R, RECON, CBC, 0, true>(acc, gauge, in, g, cb, s, p, bc);
    hop<R, RECON, CBC, 0, false>(acc, gauge, in, g, cb, s, p, bc);
    hop<R, RECON, CBC, 1, true>(acc, gauge, in, g, cb, s, p, bc);
    hop<R, RECON, CBC, 1, false>(acc, gauge, in, g, cb, s, p, bc);
    hop<R, RECON, CBC, 2, true>(acc, gauge, in, g, cb, s, p, bc);
    hop<R, RECON, CBC, 2, false>(acc, gauge, in, g, cb, s, p, bc);
    hop<R, RECON, CBC, 3, true>(acc, gauge, in, g, cb, s, p, bc);
    hop<R, RECON, CBC, 3, false>(acc, gauge, in, g, cb, s, p, bc);

    if (XPAY) {
        R x[24];
        load_spinor<R>(xin, g.Vh, cb, x);
#pragma unroll
        for (int k = 0; k < 24; ++k) acc[k] = x[k] + a * acc[k];
    }
    store_spinor<R>(out, g.Vh, cb, acc);
}

}  // namespace lqcd
