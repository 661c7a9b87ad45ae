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
// with no accepted attempt is left alone).
//
// Layout: the "update layout" of the link field, structure of arrays and checkerboarded like the spinors of the dslash:
//   double2 word w = 3 row + col of U_mu(x), x of parity p and checkerboard index cb, at
//   ((mu 2 + p) 9 + w) Vp + cb,   Vp = 32 ntiles (sites per parity, padded to whole tiles)
// so the 32 lanes of a warp read one word of 32 consecutive sites as one 512-byte run, for the thread's own link and
// (up to lattice wrap-arounds) for each of the 18 staple links.  lqcd_pack_update_links / lqcd_unpack_update_links
// convert from / to the canonical [mu][T][Z][Y][X][3][3] complex128 field.  fp64 only.  Links are periodic and carry no
// boundary phase.
#pragma once
#include "fields.cuh"
#include "geometry.cuh"

namespace lqcd {

constexpr int HB_BLOCK = 128;
// resident blocks per SM promised to ptxas for the heatbath kernel (register budget 65536 / (128 x value))
#ifndef LQCD_HB_MINB
#define LQCD_HB_MINB 4
#endif

struct Mat3 { double re[9], im[9]; };   // row-major: element (r, c) at 3 r + c

// word 0 of U_mu(x) for x = (parity p, checkerboard index cb); word w is w Vp further on
__host__ __device__ __forceinline__ size_t update_word0(int ntiles, int mu, int p, int cb) {
    return (size_t)((mu * 2 + p) * 9) * ((size_t)TILE * ntiles) + cb;
}
// RO: the link is not written by the running launch (every link but the thread's own): read-only path
template <bool RO = true>
__device__ __forceinline__ void load_mat(const double2* links, int ntiles, int mu, int p, int cb, Mat3& m) {
    const double2* q = links + update_word0(ntiles, mu, p, cb);
    const size_t Vp = (size_t)TILE * ntiles;
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        const double2 z = RO ? __ldg(q + k * Vp) : q[k * Vp];
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

// Register-lean forms of the staple products (five live 3x3 complex matrices are 180 registers; these keep at most
// three): the left / right operand is streamed from memory row by row instead of being held whole.
//   t = op(A) m2^+  with A read from memory: row r of op(A) (a column of A if ADJA) is loaded, used, dropped
template <bool ADJA>
__device__ __forceinline__ void mul_streamA_adjB(const double2* links, int ntiles, int mu, int p, int cb, const Mat3& m2, Mat3& t) {
    const double2* q = links + update_word0(ntiles, mu, p, cb);
    const size_t Vp = (size_t)TILE * ntiles;
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        double ar[3], ai[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const double2 z = __ldg(q + (ADJA ? 3 * k + r : 3 * r + k) * Vp);
            ar[k] = z.x;
            ai[k] = ADJA ? -z.y : z.y;
        }
#pragma unroll
        for (int s2 = 0; s2 < 3; ++s2) {
            double xr = 0.0, xi = 0.0;
#pragma unroll
            for (int k = 0; k < 3; ++k) {   // times conj(m2[s2][k])
                const double br = m2.re[3 * s2 + k], bi = -m2.im[3 * s2 + k];
                xr = fma(ar[k], br, xr); xr = fma(-ai[k], bi, xr);
                xi = fma(ar[k], bi, xi); xi = fma(ai[k], br, xi);
            }
            t.re[3 * r + s2] = xr;
            t.im[3 * r + s2] = xi;
        }
    }
}
//   a += t op(B)  with B read from memory: column s of op(B) (a row of B if ADJB) is loaded, used, dropped
template <bool ADJB>
__device__ __forceinline__ void addmul_streamB(Mat3& a, const Mat3& t, const double2* links, int ntiles, int mu, int p, int cb) {
    const double2* q = links + update_word0(ntiles, mu, p, cb);
    const size_t Vp = (size_t)TILE * ntiles;
#pragma unroll
    for (int s2 = 0; s2 < 3; ++s2) {
        double br[3], bi[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const double2 z = __ldg(q + (ADJB ? 3 * s2 + k : 3 * k + s2) * Vp);
            br[k] = z.x;
            bi[k] = ADJB ? -z.y : z.y;
        }
#pragma unroll
        for (int r = 0; r < 3; ++r) {
            double xr = a.re[3 * r + s2], xi = a.im[3 * r + s2];
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                xr = fma(t.re[3 * r + k], br[k], xr); xr = fma(-t.im[3 * r + k], bi[k], xr);
                xi = fma(t.re[3 * r + k], bi[k], xi); xi = fma(t.im[3 * r + k], br[k], xi);
            }
            a.re[3 * r + s2] = xr;
            a.im[3 * r + s2] = xi;
        }
    }
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

// links: update layout, updated in place for (mu, parity); uniforms: [V/2][3][4 ntries + 2]
__global__ void __launch_bounds__(HB_BLOCK, LQCD_HB_MINB) heatbath_kernel(double2* links, Geom g, double beta, int mu, int parity,
                                                                          const double* __restrict__ uniforms, int ntries) {
    const int cb = blockIdx.x * HB_BLOCK + threadIdx.x;
    if (cb >= g.Vh) return;
    const int p = parity, q = 1 - parity, nt = g.ntiles;
    const Site s = decode_site(g, cb, p);
    const int xmu = neighbour_rt(g, cb, s, 2 * mu);               // x + mu^, a site of parity q
    const Site smu = decode_site(g, xmu, q);
    Mat3 a;
#pragma unroll
    for (int k = 0; k < 9; ++k) a.re[k] = a.im[k] = 0.0;
    // the links read here belong to other sublattices (other directions, or direction mu on sites of the other parity):
    // nothing this launch writes
    for (int nu = 0; nu < 4; ++nu) {
        if (nu == mu) continue;
        Mat3 m2, t;
        // upper staple  U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+
        load_mat(links, nt, mu, q, neighbour_rt(g, cb, s, 2 * nu), m2);
        mul_streamA_adjB<false>(links, nt, nu, q, xmu, m2, t);
        addmul_streamB<true>(a, t, links, nt, nu, p, cb);
        // lower staple  U_nu(x+mu-nu)^+ U_mu(x-nu)^+ U_nu(x-nu)
        const int xdn = neighbour_rt(g, cb, s, 2 * nu + 1);       // x - nu^, parity q
        load_mat(links, nt, mu, q, xdn, m2);
        mul_streamA_adjB<true>(links, nt, nu, p, neighbour_rt(g, xmu, smu, 2 * nu + 1), m2, t);   // x + mu^ - nu^, parity p
        addmul_streamB<false>(a, t, links, nt, nu, q, xdn);
    }
    Mat3 u;
    load_mat<false>(links, nt, mu, p, cb, u);
    const double* r = uniforms + (size_t)cb * 3 * (4 * ntries + 2);
    subgroup_step<0, 1>(u, a, beta, r, ntries);
    subgroup_step<0, 2>(u, a, beta, r + (4 * ntries + 2), ntries);
    subgroup_step<1, 2>(u, a, beta, r + 2 * (4 * ntries + 2), ntries);
    double2* out = links + update_word0(nt, mu, p, cb);
    const size_t Vp = (size_t)TILE * nt;
#pragma unroll
    for (int k = 0; k < 9; ++k) out[k * Vp] = make_double2(u.re[k], u.im[k]);
}

// partial[blockIdx.y gridDim.x + blockIdx.x] = sum over the block's sites of parity blockIdx.y of the 6 Re tr U_p
__global__ void __launch_bounds__(HB_BLOCK) plaquette_kernel(const double2* __restrict__ links, Geom g, double* __restrict__ partial) {
    const int cb = blockIdx.x * HB_BLOCK + threadIdx.x, p = blockIdx.y, q = 1 - p, nt = g.ntiles;
    double sum = 0.0;
    if (cb < g.Vh) {
        const Site s = decode_site(g, cb, p);
        for (int mu = 0; mu < 4; ++mu)
            for (int nu = mu + 1; nu < 4; ++nu) {
                Mat3 m1, m2, t;
                load_mat(links, nt, mu, p, cb, m1);
                load_mat(links, nt, nu, q, neighbour_rt(g, cb, s, 2 * mu), m2);
                mul<false, false>(m1, m2, t);
                load_mat(links, nt, mu, q, neighbour_rt(g, cb, s, 2 * nu), m1);
                mul<false, true>(t, m1, m2);
                load_mat(links, nt, nu, p, cb, m1);
                // Re tr(m2 m1^+) = sum_rc Re(m2_rc conj(m1_rc))
#pragma unroll
                for (int k = 0; k < 9; ++k) sum += m2.re[k] * m1.re[k] + m2.im[k] * m1.im[k];
            }
    }
    __shared__ double warp_sums[HB_BLOCK / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, o);
    if ((threadIdx.x & 31) == 0) warp_sums[threadIdx.x >> 5] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int w = 0; w < HB_BLOCK / 32; ++w) tot += warp_sums[w];
        partial[blockIdx.y * gridDim.x + blockIdx.x] = tot;
    }
}

// Reunitarisation (reading F8), in place on the update layout; grid (ceil(Vh / block), 4 directions, 2 parities),
// one link per thread:  row0 /= |row0|;  row1 -= <row0, row1> row0, /= |row1|;  row2 = conj(row0 x row1).
__global__ void __launch_bounds__(HB_BLOCK) reunitarise_kernel(double2* links, Geom g) {
    const int cb = blockIdx.x * HB_BLOCK + threadIdx.x;
    if (cb >= g.Vh) return;
    double2* w = links + update_word0(g.ntiles, blockIdx.y, blockIdx.z, cb);
    const size_t Vp = (size_t)TILE * g.ntiles;
    double2 a[3], b[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) { a[k] = w[k * Vp]; b[k] = w[(3 + k) * Vp]; }
    double n = 0.0;
#pragma unroll
    for (int k = 0; k < 3; ++k) n += a[k].x * a[k].x + a[k].y * a[k].y;
    n = 1.0 / sqrt(n);
#pragma unroll
    for (int k = 0; k < 3; ++k) { a[k].x *= n; a[k].y *= n; }
    double pr = 0.0, pi = 0.0;   // <row0, row1> = sum conj(a_k) b_k
#pragma unroll
    for (int k = 0; k < 3; ++k) { pr += a[k].x * b[k].x + a[k].y * b[k].y; pi += a[k].x * b[k].y - a[k].y * b[k].x; }
    n = 0.0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        b[k].x -= pr * a[k].x - pi * a[k].y;
        b[k].y -= pr * a[k].y + pi * a[k].x;
        n += b[k].x * b[k].x + b[k].y * b[k].y;
    }
    n = 1.0 / sqrt(n);
#pragma unroll
    for (int k = 0; k < 3; ++k) { b[k].x *= n; b[k].y *= n; }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const int i = (k + 1) % 3, j = (k + 2) % 3;   // (a x b)_k = a_i b_j - a_j b_i, then conjugated
        const double cr = (a[i].x * b[j].x - a[i].y * b[j].y) - (a[j].x * b[i].x - a[j].y * b[i].y);
        const double ci = (a[i].x * b[j].y + a[i].y * b[j].x) - (a[j].x * b[i].y + a[j].y * b[i].x);
        w[k * Vp] = a[k];
        w[(3 + k) * Vp] = b[k];
        w[(6 + k) * Vp] = make_double2(cr, -ci);
    }
}

// canonical [mu][V][3][3] complex128 <-> update layout; grid (ceil(Vh / block), 4 directions, 2 parities)
template <bool UNPACK>
__global__ void __launch_bounds__(HB_BLOCK) update_links_pack_kernel(double2* native, double2* canon, Geom g) {
    const int cb = blockIdx.x * HB_BLOCK + threadIdx.x;
    if (cb >= g.Vh) return;
    const int mu = blockIdx.y, p = blockIdx.z;
    const Site s = decode_site(g, cb, p);
    const size_t lex = (size_t)2 * cb + s.x_odd, V = (size_t)2 * g.Vh, Vp = (size_t)TILE * g.ntiles;
    double2* c = canon + (mu * V + lex) * 9;
    double2* n = native + update_word0(g.ntiles, mu, p, cb);
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        if (UNPACK) c[k] = n[k * Vp]; else n[k * Vp] = c[k];
    }
}

}  // namespace lqcd
