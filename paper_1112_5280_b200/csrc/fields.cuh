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

__device__ __forceinline__ float fmar(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fmar(double a, double b, double c) { return fma(a, b, c); }

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

// K2: rebuild row 2 of u[18] (row-major 3x3 complex, u[6 row + 2 col + reim]) as conj(row0 x row1);
// valid for det U = +1 ("RECONSTRUCT TWELVE").
template <typename R>
__device__ __forceinline__ void recon_row2(R u[18]) {
    // row2[c] = conj(r0[a] r1[b] - r0[b] r1[a]),  (a,b) = (c+1, c+2) mod 3
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int a = (c + 1) % 3, b = (c + 2) % 3;
        const R ar = u[2 * a], ai = u[2 * a + 1], br = u[2 * b], bi = u[2 * b + 1];
        const R cr = u[6 + 2 * b], ci = u[6 + 2 * b + 1], dr = u[6 + 2 * a], di = u[6 + 2 * a + 1];
        const R re = fmar(-br, dr, fmar(bi, di, fmar(-ai, ci, ar * cr)));
        const R im = fmar(-br, di, fmar(-bi, dr, fmar(ai, cr, ar * ci)));
        u[12 + 2 * c] = re;
        u[12 + 2 * c + 1] = -im;
    }
}

// Address of word 0 of link (par, mu, cb); word w is Vh words further on.
template <typename R, int RECON>
__device__ __forceinline__ const typename LinkWord<R, RECON>::type* link_ptr(const R* __restrict__ gauge, int Vh,
                                                                             int par, int mu, int cb) {
    constexpr int NW = RECON / LinkWord<R, RECON>::LW;
    return reinterpret_cast<const typename LinkWord<R, RECON>::type*>(gauge) + (size_t)((par * 4 + mu) * NW) * Vh + cb;
}

// L1: direct (register) link load + K2.
template <typename R, int RECON>
__device__ __forceinline__ void load_link(const R* __restrict__ gauge, int Vh, int par, int mu, int cb, R u[18]) {
    using LWd = typename LinkWord<R, RECON>::type;
    constexpr int LW = LinkWord<R, RECON>::LW, NW = RECON / LW;
    const LWd* p = link_ptr<R, RECON>(gauge, Vh, par, mu, cb);
#pragma unroll
    for (int w = 0; w < NW; ++w) {
        LWd x = ld_stream(p + (size_t)w * Vh);
        unpack(x, u + w * LW);
    }
    if constexpr (RECON == 12) recon_row2<R>(u);
}

// L1, staged: each thread streams its own links into shared memory with cp.async (LDGSTS) DEPTH hops
// ahead of their use, so the DRAM-bound 2/3 of the traffic is in flight without holding registers.
// A thread only ever reads back the words it copied itself, so no block-level barrier is needed:
// cp.async.wait_group orders the copy before the read.  Slot layout [slot][word][thread], 16-byte
// (8-byte for fp32 18-real) words: conflict-free for a warp.
__device__ __forceinline__ void cp_async_word(float4* dst, const float4* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_word(double2* dst, const double2* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_word(float2* dst, const float2* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <typename R, int RECON, int BLOCK, int DEPTH>
struct LinkStage {
    using LWd = typename LinkWord<R, RECON>::type;
    static constexpr int LW = LinkWord<R, RECON>::LW, NW = RECON / LW;
    static constexpr size_t BYTES = (size_t)DEPTH * NW * BLOCK * sizeof(LWd);
    LWd* mine;  // this thread's word 0 of slot 0

    __device__ __forceinline__ explicit LinkStage(void* smem) : mine(static_cast<LWd*>(smem) + threadIdx.x) {}

    // start the copy of one link into the slot of hop k, as one commit group
    __device__ __forceinline__ void issue(int k, const LWd* src, int Vh) {
        LWd* d = mine + (k % DEPTH) * NW * BLOCK;
#pragma unroll
        for (int w = 0; w < NW; ++w) cp_async_word(d + w * BLOCK, src + (size_t)w * Vh);
        cp_async_commit();
    }

    // read hop k's link back (after cp_async_wait) and rebuild row 2
    __device__ __forceinline__ void read(int k, R u[18]) const {
        const LWd* d = mine + (k % DEPTH) * NW * BLOCK;
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            LWd x = d[w * BLOCK];
            unpack(x, u + w * LW);
        }
        if constexpr (RECON == 12) recon_row2<R>(u);
    }
};

}  // namespace lqcd
