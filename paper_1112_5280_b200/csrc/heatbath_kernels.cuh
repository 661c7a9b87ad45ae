// heatbath_kernels.cuh -- pure-gauge SU(3) heatbath (next row f4, last clause): "On the PGT side we need a SU(3)
// heatbath algorithm [20]" (ref. [20] at :156: Creutz, Cabibbo-Marinari, Kennedy-Pendleton; the heatbath
// is the task the paper runs beside the inverter).  DESIGN.md reading F7 fixes what the paper leaves open.
//
//   S = beta sum_p (1 - 1/3 Re tr U_p);  the part of S containing U_mu(x) is -(beta/3) Re tr(U_mu(x) A_mu(x)) with the
//   staple sum  A_mu(x) = sum_{nu != mu} [ U_nu(x+mu^) U_mu(x+nu^)^+ U_nu(x)^+ + U_nu(x+mu^-nu^)^+ U_mu(x-nu^)^+ U_nu(x-nu^) ]
//
// One launch updates the links U_mu(x) of one direction on the sites of one parity (they do not see each other through
// the action); one thread per link: six staples (12 products of 3x3 matrices, 18 gathered links), then the three
// Cabibbo-Marinari subgroup steps (0,1), (0,2), (1,2), each drawing its SU(2) element with the Kennedy-Pendleton
// sampler from uniforms the CALLER supplies (uniforms[cb][subgroup][4 ntries + 2]; at most ntries attempts, a subgroup
// with no accepted attempt is left alone).  Works on the canonical link field [mu][T][Z][Y][X][3][3] complex128 in
// place: a link is 144 contiguous bytes, so even the every-other-site access of a checkerboard wastes only the sectors
// at the seams, and the repack for the dslash kernels (lqcd_pack_gauge) is needed once per configuration anyway.
// fp64 only.  Links are periodic and carry no boundary phase.
#pragma once
#include "geometry.cuh"

namespace lqcd {

constexpr int HB_BLOCK = 128;
// resident blocks per SM promised to ptxas for the heatbath kernel (register budget 65536 / (128 x value))
#ifndef LQCD_HB_MINB
#define LQCD_HB_MINB 3
#endif

struct Mat3 { double re[9], im[9]; };   // row-major: element (r, c) at 3 r + c

// RO: the link is not written by the running launch (every link but the thread's own): read-only path
template <bool RO = true>
__device__ __forceinline__ void load_mat(const double* links, size_t link, Mat3& m) {
    const double2* p = reinterpret_cast<const double2*>(links) + link * 9;
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        const double2 z = RO ? __ldg(p + k) : p[k];
        m.re[k] = z.x;
        m.im[k] = z.y;
    }
}

// c = a b,  a b^+,  a^+ b  (OPA / OPB: take the adjoint of that operand)
template <bool ADJA, bool ADJB>
__device__ __forceinline__ void mul(const Mat3& a, const Mat3& b, Mat3& c) {
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int s = 0; s < 3; ++s) {
            double xr = 0.0, xi = 0.0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const int ia = ADJA ? 3 * k + r : 3 * r + k, ib = ADJB ? 3 * s + k : 3 * k + s;
                const double ar = a.re[ia], ai = ADJA ? -a.im[ia] : a.im[ia];
                const double br = b.re[ib], bi = ADJB ? -b.im[ib] : b.im[ib];
                xr = fma(ar, br, xr); xr = fma(-ai, bi, xr);
                xi = fma(ar, bi, xi); xi = fma(ai, br, xi);
            }
            c.re[3 * r + s] = xr;
            c.im[3 * r + s] = xi;
        }
}

// coordinates of a site and its lexicographic index; run-time directions are resolved with selects, not indexed arrays
// (which would live in local memory)
struct Coords { int c0, c1, c2, c3; size_t lex; };
__device__ __forceinline__ int coord(const Coords& c, int mu) { return mu == 0 ? c.c0 : (mu == 1 ? c.c1 : (mu == 2 ? c.c2 : c.c3)); }
__device__ __forceinline__ int extent(const Geom& g, int mu) { return mu == 0 ? g.X : (mu == 1 ? g.Y : (mu == 2 ? g.Z : g.T)); }
__device__ __forceinline__ long long stride(const Geom& g, int mu) {
    return mu == 0 ? 1 : (mu == 1 ? g.X : (mu == 2 ? (long long)g.X * g.Y : (long long)g.X * g.Y * g.Z));
}
// lexicographic index of the site one step (d = +1 / -1) along mu from c, periodic
__device__ __forceinline__ size_t hop(const Geom& g, const Coords& c, size_t lex, int mu, int d) {
    const int x = coord(c, mu), L = extent(g, mu);
    const long long st = stride(g, mu);
    if (d > 0) return x == L - 1 ? lex - (size_t)((L - 1) * st) : lex + (size_t)st;
    return x == 0 ? lex + (size_t)((L - 1) * st) : lex - (size_t)st;
}

// One Cabibbo-Marinari step in the block (I, J) on the link u with staple sum a: u <- G u.
template <int I, int J>
__device__ __forceinline__ void subgroup_step(Mat3& u, const Mat3& a, double beta, const double* __restrict__ r, int ntries) {
    // rows I, J of W = u a are all the step needs
    double wr[2][3], wi[2][3];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const int row = q == 0 ? I : J;
#pragma unroll
        for (int s = 0; s < 3; ++s) {
            double xr = 0.0, xi = 0.0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                xr = fma(u.re[3 * row + k], a.re[3 * k + s], xr); xr = fma(-u.im[3 * row + k], a.im[3 * k + s], xr);
                xi = fma(u.re[3 * row + k], a.im[3 * k + s], xi); xi = fma(u.im[3 * row + k], a.re[3 * k + s], xi);
            }
            wr[q][s] = xr;
            wi[q][s] = xi;
        }
    }
    // the SU(2)-proportional part of the block [[W_II, W_IJ], [W_JI, W_JJ]]:  v0 + i sigma.v
    const double v0 = 0.5 * (wr[0][I] + wr[1][J]), v3 = 0.5 * (wi[0][I] - wi[1][J]);
    const double v1 = 0.5 * (wi[0][J] + wi[1][I]), v2 = 0.5 * (wr[0][J] - wr[1][I]);
    const double k = sqrt(v0 * v0 + v1 * v1 + v2 * v2 + v3 * v3);
    const double alpha = 2.0 * beta * k / 3.0;
    // Kennedy-Pendleton: a0 with density sqrt(1 - a0^2) exp(alpha a0)
    double a0 = 1.0;
    bool accepted = false;
    for (int t = 0; t < ntries && !accepted; ++t) {
        const double r1 = r[4 * t], r2 = r[4 * t + 1], r3 = r[4 * t + 2], r4 = r[4 * t + 3];
        const double c = cos(2.0 * 3.14159265358979323846 * r2);
        const double lam2 = -(log(r1) + c * c * log(r3)) / (2.0 * alpha);
        if (r4 * r4 <= 1.0 - lam2) {
            a0 = 1.0 - 2.0 * lam2;
            accepted = true;
        }
    }
    if (!accepted) return;
    const double s = sqrt(fmax(1.0 - a0 * a0, 0.0));
    const double ct = 2.0 * r[4 * ntries] - 1.0, st = sqrt(fmax(1.0 - ct * ct, 0.0));
    double sp, cp;
    sincos(2.0 * 3.14159265358979323846 * r[4 * ntries + 1], &sp, &cp);
    const double a1 = s * st * cp, a2 = s * st * sp, a3 = s * ct;
    // g = a vbar / k  (quaternion product, vbar = v0 - i sigma.v)
    const double b0 = v0 / k, b1 = -v1 / k, b2 = -v2 / k, b3 = -v3 / k;
    const double g0 = a0 * b0 - a1 * b1 - a2 * b2 - a3 * b3;
    const double g1 = a0 * b1 + a1 * b0 - (a2 * b3 - a3 * b2);
    const double g2 = a0 * b2 + a2 * b0 - (a3 * b1 - a1 * b3);
    const double g3 = a0 * b3 + a3 * b0 - (a1 * b2 - a2 * b1);
    // G = [[g0 + i g3, g2 + i g1], [-g2 + i g1, g0 - i g3]] in rows / columns I, J:  rows I, J of u <- G (rows I, J of u)
#pragma unroll
    for (int c2 = 0; c2 < 3; ++c2) {
        const double ur = u.re[3 * I + c2], ui = u.im[3 * I + c2], vr = u.re[3 * J + c2], vi = u.im[3 * J + c2];
        u.re[3 * I + c2] = g0 * ur - g3 * ui + g2 * vr - g1 * vi;
        u.im[3 * I + c2] = g0 * ui + g3 * ur + g2 * vi + g1 * vr;
        u.re[3 * J + c2] = -g2 * ur - g1 * ui + g0 * vr + g3 * vi;
        u.im[3 * J + c2] = -g2 * ui + g1 * ur + g0 * vi - g3 * vr;
    }
}

__device__ __forceinline__ Coords site_coords(const Geom& g, int cb, int parity) {
    const Site s = decode_site(g, cb, parity);
    Coords c;
    c.c0 = 2 * s.xh + s.x_odd; c.c1 = s.y; c.c2 = s.z; c.c3 = s.t;
    c.lex = (size_t)2 * cb + s.x_odd;
    return c;
}

// links: canonical [mu][V][3][3] complex128, updated in place for (mu, parity); uniforms: [V/2][3][4 ntries + 2]
__global__ void __launch_bounds__(HB_BLOCK, LQCD_HB_MINB) heatbath_kernel(double* links, Geom g, double beta, int mu, int parity,
                                                            const double* __restrict__ uniforms, int ntries) {
    const int cb = blockIdx.x * HB_BLOCK + threadIdx.x;
    if (cb >= g.Vh) return;
    const Coords c = site_coords(g, cb, parity);
    const size_t V = (size_t)2 * g.Vh;
    const size_t x0 = c.lex, xmu = hop(g, c, x0, mu, +1);
    Mat3 a;
#pragma unroll
    for (int k = 0; k < 9; ++k) a.re[k] = a.im[k] = 0.0;
    // the links read here belong to other sublattices (other directions, or direction mu on sites of the other parity):
    // nothing this launch writes
    for (int nu = 0; nu < 4; ++nu) {
        if (nu == mu) continue;
        Mat3 p, q, t;
        // upper staple  U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+
        load_mat(links, nu * V + xmu, p);
        load_mat(links, mu * V + hop(g, c, x0, nu, +1), q);
        mul<false, true>(p, q, t);
        load_mat(links, nu * V + x0, p);
        mul<false, true>(t, p, q);
#pragma unroll
        for (int k = 0; k < 9; ++k) { a.re[k] += q.re[k]; a.im[k] += q.im[k]; }
        // lower staple  U_nu(x+mu-nu)^+ U_mu(x-nu)^+ U_nu(x-nu)
        const size_t xdn = hop(g, c, x0, nu, -1);
        load_mat(links, nu * V + hop(g, c, xmu, nu, -1), p);   // x + mu^ - nu^: the nu coordinate of x + mu^ is that of x
        load_mat(links, mu * V + xdn, q);
        mul<true, true>(p, q, t);
        load_mat(links, nu * V + xdn, p);
        mul<false, false>(t, p, q);
#pragma unroll
        for (int k = 0; k < 9; ++k) { a.re[k] += q.re[k]; a.im[k] += q.im[k]; }
    }
    Mat3 u;
    load_mat<false>(links, mu * V + x0, u);
    const double* r = uniforms + (size_t)cb * 3 * (4 * ntries + 2);
    subgroup_step<0, 1>(u, a, beta, r, ntries);
    subgroup_step<0, 2>(u, a, beta, r + (4 * ntries + 2), ntries);
    subgroup_step<1, 2>(u, a, beta, r + 2 * (4 * ntries + 2), ntries);
    double2* out = reinterpret_cast<double2*>(links) + (mu * V + x0) * 9;
#pragma unroll
    for (int k = 0; k < 9; ++k) out[k] = make_double2(u.re[k], u.im[k]);
}

// partial[block] = sum over the block's sites (both parities: thread = lexicographic site) of the 6 Re tr U_p
__global__ void __launch_bounds__(HB_BLOCK) plaquette_kernel(const double* __restrict__ links, Geom g, double* __restrict__ partial) {
    const size_t V = (size_t)2 * g.Vh;
    const size_t lex = (size_t)blockIdx.x * HB_BLOCK + threadIdx.x;
    double s = 0.0;
    if (lex < V) {
        Coords c;
        size_t r = lex;
        c.c0 = (int)(r % g.X); r /= g.X;
        c.c1 = (int)(r % g.Y); r /= g.Y;
        c.c2 = (int)(r % g.Z); c.c3 = (int)(r / g.Z);
        c.lex = lex;
        for (int mu = 0; mu < 4; ++mu)
            for (int nu = mu + 1; nu < 4; ++nu) {
                Mat3 p, q, t;
                load_mat(links, mu * V + lex, p);
                load_mat(links, nu * V + hop(g, c, lex, mu, +1), q);
                mul<false, false>(p, q, t);
                load_mat(links, mu * V + hop(g, c, lex, nu, +1), p);
                mul<false, true>(t, p, q);
                load_mat(links, nu * V + lex, p);
                // Re tr(q p^+) = sum_rc Re(q_rc conj(p_rc))
#pragma unroll
                for (int k = 0; k < 9; ++k) s += q.re[k] * p.re[k] + q.im[k] * p.im[k];
            }
    }
    __shared__ double warp_sums[HB_BLOCK / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) warp_sums[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int w = 0; w < HB_BLOCK / 32; ++w) tot += warp_sums[w];
        partial[blockIdx.x] = tot;
    }
}

}  // namespace lqcd
