// blas_kernels.cuh -- vector updates and reductions of the CG solver (next row f2; "the inversion of the
// fermion matrix"), on native half spinors (fields.cuh), one thread per site.
//
// All scalars of the iteration (alpha, beta, <r,r>, the convergence flag, the iteration count) live in device
// memory: the update kernels read them there and the loop never waits for the host except for an occasional
// look at the flag.  Reductions are deterministic: per-block partial sums in double, then one block adds the
// partials in a fixed order.  Once `done` is set, the update kernels leave x, r and p untouched, so the
// iterations the host enqueues before it notices are harmless.
#pragma once
#include "fields.cuh"
#include "geometry.cuh"

namespace lqcd {

constexpr int BLAS_BLOCK = 256;

struct CgScalars {
    double rr;     // <r, r> of the current residual
    double bb;     // <b, b>
    double alpha, beta;
    double tol2;   // tol^2
    int done;      // 1 once rr <= tol^2 bb (or b = 0)
    int iters;     // iterations performed until `done`
};

enum { CG_OP_INIT = 0, CG_OP_PAP = 1, CG_OP_RR = 2 };

// sum over the block, result valid in thread 0; fixed order (shuffle tree, then warp 0 over the warp sums)
__device__ __forceinline__ double block_sum(double v) {
    __shared__ double warp_sums[BLAS_BLOCK / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) warp_sums[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        v = threadIdx.x < BLAS_BLOCK / 32 ? warp_sums[threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    }
    return v;
}

// A site of a native half spinor as numbers of the arithmetic type A = Compute<S>::type, for any storage type S (float,
// double, or __half = 16-bit storage: 24 normalised halfs and an fp32 site norm; the store re-normalises and rounds).
// RW: the calling kernel also writes the field -- coherent loads instead of the read-only path.
template <typename S, bool RW>
__device__ __forceinline__ void load_vec(const S* base, int ntiles, int cb, typename Compute<S>::type v[24]) {
    if constexpr (sizeof(S) == 2) {
        float n;
        if constexpr (RW) load_spinor_h_rw(base, ntiles, cb, v, n); else load_spinor_h(base, ntiles, cb, v, n);
#pragma unroll
        for (int k = 0; k < 24; ++k) v[k] *= n;
    } else if constexpr (RW) {
        load_spinor_rw<S>(base, cb, v);
    } else {
        load_spinor<S>(base, cb, v);
    }
}

template <typename R>
__device__ __forceinline__ double site_norm2(const R v[24]) {
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 24; ++k) s += (double)v[k] * (double)v[k];
    return s;
}

// partial[blockIdx.x] = sum over the block's sites of |v(x)|^2
template <typename S>
__global__ void __launch_bounds__(BLAS_BLOCK) norm2_kernel(const S* __restrict__ v, Geom g, double* __restrict__ partial) {
    using A = typename Compute<S>::type;
    const int cb = blockIdx.x * BLAS_BLOCK + threadIdx.x;
    double s = 0.0;
    if (cb < g.Vh) {
        A a[24];
        load_vec<S, false>(v, g.ntiles, cb, a);
        s = site_norm2<A>(a);
    }
    s = block_sum(s);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// One block: total = sum of partial[0..n) in a fixed order, then the scalar step `op` of the iteration.
__global__ void __launch_bounds__(BLAS_BLOCK) cg_scalar_kernel(const double* __restrict__ partial, int n, CgScalars* sc, int op) {
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += BLAS_BLOCK) s += partial[i];
    s = block_sum(s);
    if (threadIdx.x != 0) return;
    if (op == CG_OP_INIT) {            // s = <b, b>
        sc->bb = sc->rr = s;
        sc->alpha = sc->beta = 0.0;
        sc->iters = 0;
        sc->done = (s == 0.0);
    } else if (op == CG_OP_PAP) {      // s = <p, A p> = |Q p|^2
        sc->alpha = sc->done ? 0.0 : sc->rr / s;
    } else if (!sc->done) {            // CG_OP_RR: s = <r, r> after the update
        sc->iters += 1;
        sc->beta = s / sc->rr;
        sc->rr = s;
        if (s <= sc->tol2 * sc->bb) sc->done = 1;
    }
}

// x += alpha p;  r -= alpha s;  partial = block sums of |r|^2       (skipped once done)
// X: storage of the iterate and the residual; P: storage of the search direction and of A p (the 16-bit solver keeps
// x and r in fp32 -- their recurrences carry the accuracy -- and p, A p in the operator's 16-bit format)
template <typename X, typename P>
__global__ void __launch_bounds__(BLAS_BLOCK) cg_update_xr_kernel(X* x, X* r, const P* __restrict__ p,
                                                                   const P* __restrict__ s, Geom g, const CgScalars* __restrict__ sc,
                                                                   double* __restrict__ partial) {
    using A = typename Compute<X>::type;
    const int cb = blockIdx.x * BLAS_BLOCK + threadIdx.x;
    const bool done = sc->done != 0;
    const A alpha = (A)sc->alpha;
    double n2 = 0.0;
    if (cb < g.Vh) {
        A rv[24];
        load_vec<X, true>(r, g.ntiles, cb, rv);   // r and x are updated in place: coherent loads, not .nc
        if (!done) {
            A xv[24];
            typename Compute<P>::type pv[24], sv[24];
            load_vec<X, true>(x, g.ntiles, cb, xv);
            load_vec<P, false>(p, g.ntiles, cb, pv);
            load_vec<P, false>(s, g.ntiles, cb, sv);
#pragma unroll
            for (int k = 0; k < 24; ++k) {
                xv[k] = fmar(alpha, (A)pv[k], xv[k]);
                rv[k] = fmar(-alpha, (A)sv[k], rv[k]);
            }
            store_field<X>(x, g.ntiles, cb, xv);
            store_field<X>(r, g.ntiles, cb, rv);
        }
        n2 = site_norm2<A>(rv);
    }
    n2 = block_sum(n2);
    if (threadIdx.x == 0) partial[blockIdx.x] = n2;
}

// p = r + beta p       (skipped once done)
template <typename X, typename P>
__global__ void __launch_bounds__(BLAS_BLOCK) cg_update_p_kernel(P* p, const X* __restrict__ r, Geom g,
                                                                  const CgScalars* __restrict__ sc) {
    using A = typename Compute<P>::type;
    const int cb = blockIdx.x * BLAS_BLOCK + threadIdx.x;
    if (cb >= g.Vh || sc->done) return;
    const A beta = (A)sc->beta;
    A pv[24];
    typename Compute<X>::type rv[24];
    load_vec<P, true>(p, g.ntiles, cb, pv);   // p is updated in place
    load_vec<X, false>(r, g.ntiles, cb, rv);
#pragma unroll
    for (int k = 0; k < 24; ++k) pv[k] = fmar(beta, pv[k], (A)rv[k]);
    store_field<P>(p, g.ntiles, cb, pv);
}

// ---- mixed-precision defect correction (fp64 outer, fp32 inner CG) -------------------------------------

// dst = src converted to dst's storage type, site by site (the formats have different words per site in the native layout)
template <typename Sd, typename Ss>
__global__ void __launch_bounds__(BLAS_BLOCK) convert_kernel(Sd* __restrict__ dst, const Ss* __restrict__ src, Geom g) {
    const int cb = blockIdx.x * BLAS_BLOCK + threadIdx.x;
    if (cb >= g.Vh) return;
    typename Compute<Ss>::type a[24];
    typename Compute<Sd>::type b[24];
    load_vec<Ss, false>(src, g.ntiles, cb, a);
#pragma unroll
    for (int k = 0; k < 24; ++k) b[k] = (typename Compute<Sd>::type)a[k];
    store_field<Sd>(dst, g.ntiles, cb, b);
}

// x += (double) e
__global__ void __launch_bounds__(BLAS_BLOCK) accumulate_correction_kernel(double* x, const float* __restrict__ e, Geom g) {
    const int cb = blockIdx.x * BLAS_BLOCK + threadIdx.x;
    if (cb >= g.Vh) return;
    double xv[24];
    float ev[24];
    load_spinor_rw<double>(x, cb, xv);   // x is updated in place
    load_spinor<float>(e, cb, ev);
#pragma unroll
    for (int k = 0; k < 24; ++k) xv[k] += (double)ev[k];
    store_spinor<double>(x, cb, xv);
}

// r = b - s;  partial = block sums of |r|^2
template <typename R>
__global__ void __launch_bounds__(BLAS_BLOCK) residual_kernel(R* __restrict__ r, const R* __restrict__ b, const R* __restrict__ s,
                                                               Geom g, double* __restrict__ partial) {
    const int cb = blockIdx.x * BLAS_BLOCK + threadIdx.x;
    double n2 = 0.0;
    if (cb < g.Vh) {
        R bv[24], sv[24];
        load_spinor<R>(b, cb, bv);
        load_spinor<R>(s, cb, sv);
#pragma unroll
        for (int k = 0; k < 24; ++k) bv[k] -= sv[k];
        store_spinor<R>(r, cb, bv);
        n2 = site_norm2<R>(bv);
    }
    n2 = block_sum(n2);
    if (threadIdx.x == 0) partial[blockIdx.x] = n2;
}

// One block: *out = sum of partial[0..n) in a fixed order
__global__ void __launch_bounds__(BLAS_BLOCK) sum_partials_kernel(const double* __restrict__ partial, int n, double* out) {
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += BLAS_BLOCK) s += partial[i];
    s = block_sum(s);
    if (threadIdx.x == 0) *out = s;
}

}  // namespace lqcd
