// pack_kernels.cuh -- canonical (interchange) <-> native layout conversion (step L0).
// Layout only, no arithmetic of the method; built once per field, not on the timed path.
// Layouts are specified in include/lqcd.h and fields.cuh.
#pragma once
#include "fields.cuh"
#include "geometry.cuh"

namespace lqcd {

// lex index of the site (parity p, checkerboard index cb): x = 2 xh + x_odd  =>  lex = 2 cb + x_odd.
__device__ __forceinline__ size_t lex_of(const Geom& g, int cb, int p) {
    const Site s = decode_site(g, cb, p);
    return (size_t)2 * cb + s.x_odd;
}

// lex index of the site one step back along mu from (parity p, cb), periodic wrap (links carry no phase)
__device__ __forceinline__ size_t lex_back(const Geom& g, int cb, int p, int mu) {
    const Site s = decode_site(g, cb, p);
    int c[4] = {2 * s.xh + s.x_odd, s.y, s.z, s.t};
    const int L[4] = {g.X, g.Y, g.Z, g.T};
    c[mu] = c[mu] == 0 ? L[mu] - 1 : c[mu] - 1;
    return (size_t)c[0] + (size_t)g.X * (c[1] + (size_t)g.Y * (c[2] + (size_t)g.Z * c[3]));
}

// The canonical link (18 reals) stored for hop k of the site (p, cb).  On a time slab (`below` != NULL) the backward
// t link of a site of the first slice, U_t(x - t^), belongs to the rank below and comes from `below`, a canonical
// [Z][Y][X][3][3] array of that rank's last-slice t links; everywhere else the local field with periodic wrap.
template <typename R>
__device__ __forceinline__ const R* link_source(const R* __restrict__ canon, const R* __restrict__ below, const Geom& g, int cb, int p, int k) {
    const int mu = k >> 1;
    const size_t V = (size_t)2 * g.Vh;
    if (k == 7 && below && cb < g.st) {   // t = 0
        const size_t lex = lex_of(g, cb, p);  // t = 0: lex is the index within the slice
        return below + lex * 18;
    }
    const size_t site = (k & 1) ? lex_back(g, cb, p, mu) : lex_of(g, cb, p);
    return canon + ((size_t)mu * V + site) * 18;
}

// canonical links [mu][V][3][3] complex -> native, gathered by output site (fields.cuh): for site cb of
// parity p, hop k = 2 mu holds U_mu(x), hop k = 2 mu + 1 holds U_mu(x - mu^); first RECON reals of each.
// grid: (ceil(Vh / block), 8 hops, 2 parities).
template <typename R, int RECON>
__global__ void pack_gauge_kernel(R* __restrict__ native, const R* __restrict__ canon, const R* __restrict__ below, Geom g) {
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= g.Vh) return;
    const int k = blockIdx.y, p = blockIdx.z;
    constexpr int LW = LinkWord<R, RECON>::LW, NW = RECON / LW;
    const R* src = link_source<R>(canon, below, g, cb, p, k);
    R* dst = native + link_word0<R, RECON>(g.ntiles, p, cb, k) * LW;
#pragma unroll
    for (int w = 0; w < NW; ++w)
#pragma unroll
        for (int l = 0; l < LW; ++l) dst[(size_t)w * TILE * LW + l] = src[w * LW + l];
}

// 8-real storage (fields.cuh): r = (Re a1, Im a1, Re a2, Im a2, Re b0, Im b0, arg(a0) / pi, arg(c0) / pi), the two
// phases evaluated in double and rounded once.  Same grid as pack_gauge_kernel.
template <typename R>
__global__ void pack_gauge8_kernel(R* __restrict__ native, const R* __restrict__ canon, const R* __restrict__ below, Geom g,
                                   double min_margin2, unsigned* __restrict__ bad) {
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= g.Vh) return;
    const int k = blockIdx.y, p = blockIdx.z;
    const R* src = link_source<R>(canon, below, g, cb, p, k);
    // the three squared moduli the decoder (recon8, fields.cuh) takes roots of and divides by: |U00|^2, N2 = |U01|^2 + |U02|^2,
    // |U20|^2.  A link with one of them below min_margin2 cannot be decoded (unit links: N2 = 0 -> NaN): report it.
    {
        const double a0 = (double)src[0] * src[0] + (double)src[1] * src[1];
        const double n2 = (double)src[2] * src[2] + (double)src[3] * src[3] + (double)src[4] * src[4] + (double)src[5] * src[5];
        const double c0 = (double)src[12] * src[12] + (double)src[13] * src[13];
        if (!(a0 >= min_margin2 && n2 >= min_margin2 && c0 >= min_margin2)) atomicOr(bad, 1u);   // a NaN fails every comparison
    }
    constexpr double inv_pi = 0.31830988618379067154;
    R r[8] = {src[2], src[3], src[4], src[5], src[6], src[7],
              (R)(atan2((double)src[1], (double)src[0]) * inv_pi), (R)(atan2((double)src[13], (double)src[12]) * inv_pi)};
    R* dst = native + link_word0<R, 8>(g.ntiles, p, cb, k) * 4;
#pragma unroll
    for (int w = 0; w < 2; ++w)
#pragma unroll
        for (int l = 0; l < 4; ++l) dst[(size_t)w * TILE * 4 + l] = r[w * 4 + l];
}

// min over all links of min(|a0|, sqrt(N2), |c0|)^2 -- the moduli the 8-real decoder derives from differences and
// divides by; the result is the squared margin, kept as the bit pattern of a non-negative double (ordered like
// unsigned integers) so that atomicMin applies.  grid: (ceil(4 V / block)).
template <typename R>
__global__ void recon8_margin_kernel(const R* __restrict__ canon, size_t nlinks, unsigned long long* __restrict__ out) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    double m = 1.0;
    if (i < nlinks) {
        const R* u = canon + i * 18;
        const double a0 = (double)u[0] * u[0] + (double)u[1] * u[1];
        const double n2 = (double)u[2] * u[2] + (double)u[3] * u[3] + (double)u[4] * u[4] + (double)u[5] * u[5];
        const double c0 = (double)u[12] * u[12] + (double)u[13] * u[13];
        m = fmin(a0, fmin(n2, c0));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmin(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) atomicMin(out, (unsigned long long)__double_as_longlong(m));
}

// mode 0/1: canonical half spinor [Vh][4][3] of that parity <-> native half spinor.
// mode -1 : canonical full spinor [V][4][3] <-> native full [even|odd]; blockIdx.y = parity.
template <typename R, bool UNPACK>
__global__ void pack_spinor_kernel(R* __restrict__ dst_, const R* __restrict__ src_, Geom g, int mode) {
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= g.Vh) return;
    constexpr int W = Word<R>::W, Q = 24 / W;
    size_t canon_site, native_off = 0;
    if (mode >= 0) {
        canon_site = (size_t)cb;
    } else {
        const int p = blockIdx.y;
        canon_site = lex_of(g, cb, p);
        native_off = (size_t)p * 24 * TILE * g.ntiles;
    }
    const size_t w0 = spinor_word0<R>(cb) * W;
    if (UNPACK) {
        const R* nat = src_ + native_off + w0;
        R* can = dst_ + canon_site * 24;
#pragma unroll
        for (int q = 0; q < Q; ++q)
#pragma unroll
            for (int l = 0; l < W; ++l) can[q * W + l] = nat[(size_t)q * TILE * W + l];
    } else {
        R* nat = dst_ + native_off + w0;
        const R* can = src_ + canon_site * 24;
#pragma unroll
        for (int q = 0; q < Q; ++q)
#pragma unroll
            for (int l = 0; l < W; ++l) nat[(size_t)q * TILE * W + l] = can[q * W + l];
    }
}

// ---- 16-bit storage: canonical complex64 <-> native half (fields.cuh) ------------------------------------

// 12-real links only.  grid: (ceil(Vh / block), 8 hops, 2 parities).
__global__ void pack_gauge_h_kernel(__half* __restrict__ native, const float* __restrict__ canon, const float* __restrict__ below, Geom g) {
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= g.Vh) return;
    const int k = blockIdx.y, p = blockIdx.z;
    const float* src = link_source<float>(canon, below, g, cb, p, k);
    __half* dst = native + link_word0_h(g.ntiles, p, cb, k) * 4;
#pragma unroll
    for (int w = 0; w < 3; ++w)
#pragma unroll
        for (int l = 0; l < 4; ++l) dst[(size_t)w * TILE * 4 + l] = __float2half_rn(src[w * 4 + l]);
}

// mode as in pack_spinor_kernel; the canonical side is complex64
template <bool UNPACK>
__global__ void pack_spinor_h_kernel(void* __restrict__ dst_, const void* __restrict__ src_, Geom g, int mode) {
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= g.Vh) return;
    size_t canon_site = (size_t)cb, native_off = 0;
    if (mode < 0) {
        const int p = blockIdx.y;
        canon_site = lex_of(g, cb, p);
        native_off = (size_t)p * half_stride<__half>(g.ntiles);
    }
    float v[24];
    if (UNPACK) {
        float n;
        load_spinor_h(static_cast<const __half*>(src_) + native_off, g.ntiles, cb, v, n);
        float* can = static_cast<float*>(dst_) + canon_site * 24;
#pragma unroll
        for (int k = 0; k < 24; ++k) can[k] = v[k] * n;
    } else {
        const float* can = static_cast<const float*>(src_) + canon_site * 24;
#pragma unroll
        for (int k = 0; k < 24; ++k) v[k] = can[k];
        store_spinor_h(static_cast<__half*>(dst_) + native_off, g.ntiles, cb, v);
    }
}

}  // namespace lqcd
