// pack_kernels.cuh -- canonical (interchange) <-> native layout conversion (step L0).
// Layout only, no arithmetic of the method; built once per field, not on the timed path.
// Layouts are specified in include/lqcd.h.
#pragma once
#include "fields.cuh"
#include "geometry.cuh"

namespace lqcd {

// lex index of the site (parity p, checkerboard index cb): x = 2 xh + x_odd  =>  lex = 2 cb + x_odd.
__device__ __forceinline__ size_t lex_of(const Geom& g, int cb, int p) {
    const Site s = decode_site(g, cb, p);
    return (size_t)2 * cb + s.x_odd;
}

// canonical links [mu][V][3][3] complex -> native [parity][mu][word][Vh][lane], first RECON reals.
template <typename R, int RECON>
__global__ void pack_gauge_kernel(R* __restrict__ native, const R* __restrict__ canon, Geom g) {
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= g.Vh) return;
    const int mu = blockIdx.y, p = blockIdx.z;
    constexpr int LW = LinkWord<R, RECON>::LW, NW = RECON / LW;
    const size_t V = (size_t)2 * g.Vh;
    const R* src = canon + ((size_t)mu * V + lex_of(g, cb, p)) * 18;
    R* dst = native + ((size_t)((p * 4 + mu) * NW) * g.Vh + cb) * LW;
#pragma unroll
    for (int w = 0; w < NW; ++w)
#pragma unroll
        for (int l = 0; l < LW; ++l) dst[(size_t)w * g.Vh * LW + l] = src[w * LW + l];
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
        native_off = (size_t)p * 24 * g.Vh;
    }
    if (UNPACK) {
        const R* nat = src_ + native_off;
        R* can = dst_ + canon_site * 24;
#pragma unroll
        for (int q = 0; q < Q; ++q)
#pragma unroll
            for (int l = 0; l < W; ++l) can[q * W + l] = nat[((size_t)q * g.Vh + cb) * W + l];
    } else {
        R* nat = dst_ + native_off;
        const R* can = src_ + canon_site * 24;
#pragma unroll
        for (int q = 0; q < Q; ++q)
#pragma unroll
            for (int l = 0; l < W; ++l) nat[((size_t)q * g.Vh + cb) * W + l] = can[q * W + l];
    }
}

}  // namespace lqcd
