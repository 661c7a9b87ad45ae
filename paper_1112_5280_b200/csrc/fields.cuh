// fields.cuh -- native field layout (step L0) and 128-bit loads/stores (L1, L2, L6), K2 recon.
//
// Native layout (include/lqcd.h):
//   spinor: real r = 6 spin + 2 colour + reim in [0,24); W = 16/sizeof(R) reals per word;
//           word q = r / W of site cb at word index q * Vh + cb  (consecutive sites adjacent).
//   links:  real r = 6 row + 2 col + reim over the first RECON reals; words of LW reals;
//           array [parity][mu][word][Vh].
#pragma once
#include <cuda_runtime.h>

namespace lqcd {

template <typename R> struct Word;            // 128-bit word of R
template <> struct Word<float>  { using type = float4;  static constexpr int W = 4; };
template <> struct Word<double> { using type = double2; static constexpr int W = 2; };

// Link word: 16 bytes except fp32 18-real (18 = 4.5 x 4, so 9 x float2).
template <typename R, int RECON> struct LinkWord { using type = typename Word<R>::type; static constexpr int LW = Word<R>::W; };
template <> struct LinkWord<float, 18> { using type = float2; static constexpr int LW = 2; };

__device__ __forceinline__ void unpack(const float4& w, float* v)  { v[0] = w.x; v[1] = w.y; v[2] = w.z; v[3] = w.w; }
__device__ __forceinline__ void unpack(const float2& w, float* v)  { v[0] = w.x; v[1] = w.y; }
__device__ __forceinline__ void unpack(const double2& w, double* v) { v[0] = w.x; v[1] = w.y; }
__device__ __forceinline__ float4  pack4(const float* v)  { return make_float4(v[0], v[1], v[2], v[3]); }
__device__ __forceinline__ double2 pack2(const double* v) { return make_double2(v[0], v[1]); }

// Spinor loads take the default cached path: each input spinor is gathered by 8 output
// sites, and that reuse must come from L1/L2, not from DRAM.
template <typename R>
__device__ __forceinline__ void load_spinor(const R* __restrict__ base, int Vh, int cb, R v[24]) {
    using Wd = typename Word<R>::type;
    constexpr int W = Word<R>::W, Q = 24 / W;
    const Wd* p = reinterpret_cast<const Wd*>(base) + cb;
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        Wd w = __ldg(p + (size_t)q * Vh);
        unpack(w, v + q * W);
    }
}

__device__ __forceinline__ void st_stream(float4* p, float4 v)  { __stcs(p, v); }
__device__ __forceinline__ void st_stream(double2* p, double2 v) { __stcs(p, v); }

template <typename R>
__device__ __forceinline__ void store_spinor(R* __restrict__ base, int Vh, int cb, const R v[24]) {
    using Wd = typename Word<R>::type;
    constexpr int W = Word<R>::W, Q = 24 / W;
    Wd* p = reinterpret_cast<Wd*>(base) + cb;
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        Wd w;
        if constexpr (W == 4) w = pack4(v + q * W); else w = pack2(v + q * W);
        p[(size_t)q * Vh] = w;
    }
}

// Links are read exactly once per application: streaming loads (ld.global.cs, evict-first)
// so they do not push the spinor working set out of L2.
__device__ __forceinline__ float4  ld_stream(const float4* p)  { return __ldcs(p); }
__device__ __forceinline__ float2  ld_stream(const float2* p)  { return __ldcs(p); }
__device__ __forceinline__ double2 ld_stream(const double2* p) { return __ldcs(p); }

// u[18]: row-major 3x3 complex, u[6 row + 2 col + reim].  RECON == 12 rebuilds row 2 as
// conj(row0 x row1) (K2; valid for det U = +1; "RECONSTRUCT TWELVE").
template <typename R, int RECON>
__device__ __forceinline__ void load_link(const R* __restrict__ gauge, int Vh, int par, int mu, int cb, R u[18]) {
    using LWd = typename LinkWord<R, RECON>::type;
    constexpr int LW = LinkWord<R, RECON>::LW, NW = RECON / LW;
    const LWd* p = reinterpret_cast<const LWd*>(gauge) + (size_t)((par * 4 + mu) * NW) * Vh + cb;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
        LWd x = ld_stream(p + (size_t)w * Vh);
        unpack(x, u + w * LW);
    }
    if constexpr (RECON == 12) {
        // row2[c] = conj(r0[a] r1[b] - r0[b] r1[a]),  (a,b) = (c+1, c+2) mod 3
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int a = (c + 1) % 3, b = (c + 2) % 3;
            const R ar = u[2 * a], ai = u[2 * a + 1], br = u[2 * b], bi = u[2 * b + 1];
            const R cr = u[6 + 2 * b], ci = u[6 + 2 * b + 1], dr = u[6 + 2 * a], di = u[6 + 2 * a + 1];
            // r0[a]*r1[b] - r0[b]*r1[a]
            const R re = ar * cr - ai * ci - (br * dr - bi * di);
            const R im = ar * ci + ai * cr - (br * di + bi * dr);
            u[12 + 2 * c] = re;
            u[12 + 2 * c + 1] = -im;
        }
    }
}

}  // namespace lqcd
