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

template <typename R>
__device__ __forceinline__ double site_norm2(const R v[24]) {
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 24; ++k) s += (double)v[k] * (double)v[k];
    return s;
}

// partial[blockIdx.x] = sum over the block's sites of |v(x)|^2
template <typename R>
__global__ void __launch_bounds__(BLAS_BLOCK) norm2_kernel(const R* __restrict__ v, Geom g, double* __restrict__ partial) {
    const int cb = blockIdx.x * BLAS_BLOCK + threadIdx.x;
    double s = 0.0;
    if (cb < g.Vh) {
        R a[24];
        load_spinor<R>(v, cb, a);
        s = site_norm2<R>(a);
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
template <typename R>
__global__ void __launch_bounds__(BLAS_BLOCK) cg_update_xr_kernel(R* x, R* r, const R* __restrict__ p,
                                                                   const R* __restrict__ s, Geom g, const CgScalars* __restrict__ sc,
                                                                   double* __restrict__ partial) {
    const int cb = blockIdx.x * BLAS_BLOCK + threadIdx.x;
    const bool done = sc->done != 0;
    const R alpha = (R)sc->alpha;
    double n2 = 0.0;
    if (cb < g.Vh) {
        R rv[24];
        load_spinor_rw<R>(r, cb, rv);   // r and x are updated in place: coherent loads, not .nc
        if (!done) {
            R xv[24], pv[24], sv[24];
            load_spinor_rw<R>(x, cb, xv);
            load_spinor<R>(p, cb, pv);
            load_spinor<R>(s, cb, sv);
#pragma unroll
            for (int k = 0; k < 24; ++k) {
                xv[k] = fmar(alpha, pv[k], xv[k]);
                rv[k] = fmar(-alpha, sv[k], rv[k]);
            }
            store_spinor<R>(x, cb, xv);
            store_spinor<R>(r, cb, rv);
        }
        n2 = site_norm2<R>(rv);
    }
    n2 = block_sum(n2);
    if (threadIdx.x == 0) partial[blockIdx.x] = n2;
}

// p = r + beta p       (skipped once done)
template <typename R>
__global__ void __launch_bounds__(BLAS_BLOCK) cg_update_p_kernel(R* p, const R* __restrict__ r, Geom g,
                                                                  const CgScalars* __restrict__ sc) {
    const int cb = blockIdx.x * BLAS_BLOCK + threadIdx.x;
    if (cb >= g.Vh || sc->done) return;
    const R beta = (R)sc->beta;
    R pv[24], rv[24];
    load_spinor_rw<R>(p, cb, pv);   // p is updated in place
    load_spinor<R>(r, cb, rv);
#pragma unroll
    for (int k = 0; k < 24; ++k) pv[k] = fmar(beta, pv[k], rv[k]);
    store_spinor<R>(p, cb, pv);
}

// ---- mixed-precision defect correction (fp64 outer, fp32 inner CG) -------------------------------------

// dst = (Rd) src, site by site (the two precisions have different words per site in the native layout)
template <typename Rd, typename Rs>
__global__ void __launch_bounds__(BLAS_BLOCK) convert_kernel(Rd* __restrict__ dst, const Rs* __restrict__ src, Geom g) {
    const int cb = blockIdx.x * BLAS_BLOCK + threadIdx.x;
    if (cb >= g.Vh) return;
    Rs a[24];
    Rd b[24];
    load_spinor<Rs>(src, cb, a);
#pragma unroll
    for (int k = 0; k < 24; ++k) b[k] = (Rd)a[k];
    store_spinor<Rd>(dst, cb, b);
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
