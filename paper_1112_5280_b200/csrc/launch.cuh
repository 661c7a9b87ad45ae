// launch.cuh -- host-side launch chain of the dslash kernel, shared by lqcd.cu (which only calls it) and the
// instantiation units inst_*.cu (one per storage type x link format, so that the library builds in parallel:
// each unit instantiates dslash_kernel for its 4 epilogues x 2 boundary-phase kinds).
#pragma once
#include <atomic>
#include <mutex>

#include "../../include/lqcd.h"

#include "dslash_kernel.cuh"
#include "pipe_kernel.cuh"
#include "lstage_kernel.cuh"

// streams and events of the host-buffer path (lqcd_dslash_eo_host_batch), created at its first call and kept for
// the life of the context; the mutex serialises host-path calls on one context (each call synchronises anyway)
struct lqcd_host_pipe {
    static constexpr int SLOTS = 3;
    std::mutex lock;
    bool ready = false;
    cudaStream_t up = nullptr, down = nullptr;
    cudaEvent_t start = nullptr, in_done[SLOTS] = {}, comp_done[SLOTS] = {}, out_done[SLOTS] = {};
};

struct lqcd_ctx {
    lqcd_params p;
    lqcd::Geom g;
    bool complex_bc;
    int kernel;   // LQCD_KERNEL_GATHER, _PIPE, _BLOCKED or _LSTAGE (lqcd_set_kernel)
    mutable lqcd_host_pipe host;
};

namespace lqcd {

// threads per block of the dslash kernel: 64 (two warp tiles).  128 measured the same on B200.
#ifndef LQCD_BLOCK
#define LQCD_BLOCK 64
#endif
constexpr int DSLASH_BLOCK = LQCD_BLOCK;

// counts the launch and picks up a launch error (defined in lqcd.cu)
lqcd_status after_launch();

// epilogue of one launch: mode (EPI_*) and its constants, in double until the kernel's precision is known
struct EpiArgs { int mode; double a, g_re, g_im; int g5_out; };

// range of checkerboard indices one launch covers: everything, or the time slices [t_begin, t_end)
struct CbRange { int begin, end; };

template <typename R>
BcPhases<R> make_bc(const lqcd_ctx* c) {
    BcPhases<R> b;
    for (int mu = 0; mu < 4; ++mu) {
        b.re[mu] = (R)c->p.bc_re[mu];
        b.im[mu] = (R)c->p.bc_im[mu];
    }
    return b;
}

// the pipelined kernel exists for fp32 / fp64 fields with links stored in the same precision
template <typename S, int RECON> constexpr bool pipe_capable = (sizeof(S) == 4 || sizeof(S) == 8) && (RECON == 8 || RECON == 12 || RECON == 18);

// Per-device launch state.  One process may drive several GPUs through the C ABI, so anything cached about "the device"
// is indexed by the current device's ordinal; entries are atomics because two host threads may launch at once (both then
// write the same value, which is harmless).
constexpr int MAX_DEVICES = 64;

inline int current_device() {
    int dev = -1;
    return cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < MAX_DEVICES ? dev : -1;
}

// SMs of the current device (persistent grid of the pipelined kernel); 0 on error
inline int sm_count() {
    static std::atomic<int> n[MAX_DEVICES];
    const int dev = current_device();
    if (dev < 0) return 0;
    int v = n[dev].load(std::memory_order_relaxed);
    if (v == 0 && cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess) n[dev].store(v, std::memory_order_relaxed);
    return v;
}

template <typename R, int RECON, int EPI, bool CBC>
lqcd_status launch_pipe(const lqcd_ctx* c, void* out, const void* gauge, const void* in, const void* xin,
                        const EpiArgs& e, int parity, cudaStream_t st, CbRange rg) {
    using P = Pipe<R, RECON>;
    auto kernel = dslash_pipe_kernel<R, RECON, EPI, CBC>;
    // the opt-in to more than 48 KB of dynamic shared memory is a property of the kernel ON ONE DEVICE: once per device
    static std::atomic<bool> configured[MAX_DEVICES];
    const int dev = current_device();
    if (dev < 0) return LQCD_ECUDA;
    if (!configured[dev].load(std::memory_order_acquire)) {
        if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, P::SMEM_BYTES) != cudaSuccess) return after_launch();
        configured[dev].store(true, std::memory_order_release);
    }
    const int nt = ((rg.end + TILE - 1) >> 5) - (rg.begin >> 5), nwork = parity < 0 ? 2 * nt : nt;
    const int nsm = sm_count();
    if (nsm <= 0) return LQCD_ECUDA;
    const Epilogue<R> epi{(R)e.a, (R)e.g_re, (R)e.g_im, e.g5_out};
    kernel<<<nwork < nsm ? nwork : nsm, P::THREADS, P::SMEM_BYTES, st>>>((R*)out, (const R*)gauge, (const R*)in, (const R*)xin, epi, c->g,
                                                                        parity < 0 ? 0 : parity, parity < 0 ? 1 : 0, make_bc<R>(c), rg.begin, rg.end);
    return after_launch();
}

// Box of nwarps warp tiles for the blocked map: 2 tiles along y and 2 along t where the block has the warps for it, the
// rest along z (by * bz * bt = nwarps for the warp counts in use: 16, 12, 8; other shapes were swept in round 2).
inline BlockMap box_shape(int nwarps, const Geom& g) {
    BlockMap m;
    m.ny = g.sz / TILE;
    m.by = nwarps >= 4 && m.ny >= 2 ? 2 : 1;
    m.bt = nwarps >= 8 ? 2 : 1;
    m.bz = nwarps / (m.by * m.bt);
    m.gy = (m.ny + m.by - 1) / m.by;
    m.gz = (g.Z + m.bz - 1) / m.bz;
    return m;
}

// gather kernel with the link stream staged by TMA (lstage_kernel.cuh); the range must start on a tile boundary
template <typename R, int RECON, int EPI, bool CBC>
lqcd_status launch_lstage(const lqcd_ctx* c, void* out, const void* gauge, const void* in, const void* xin,
                          const EpiArgs& e, int parity, cudaStream_t st, CbRange rg) {
    constexpr int BLOCK = DSLASH_BLOCK;
    const int smem = LStage<R, RECON>::smem_bytes(BLOCK);
    const dim3 grid((rg.end - rg.begin + BLOCK - 1) / BLOCK, parity < 0 ? 2 : 1);
    const Epilogue<R> epi{(R)e.a, (R)e.g_re, (R)e.g_im, e.g5_out};
    dslash_lstage_kernel<R, RECON, EPI, CBC, BLOCK><<<grid, BLOCK, smem, st>>>(
        (R*)out, (const R*)gauge, (const R*)in, (const R*)xin, epi, c->g, parity < 0 ? 0 : parity, make_bc<R>(c), rg.begin, rg.end);
    return after_launch();
}

template <typename S, int RECON, int EPI, bool CBC>
lqcd_status launch_one(const lqcd_ctx* c, void* out, const void* gauge, const void* in, const void* xin,
                       const EpiArgs& e, int parity, cudaStream_t st, CbRange rg) {
    if constexpr (pipe_capable<S, RECON>) {
        if (c->kernel == LQCD_KERNEL_PIPE) return launch_pipe<S, RECON, EPI, CBC>(c, out, gauge, in, xin, e, parity, st, rg);
        if (c->kernel == LQCD_KERNEL_LSTAGE && rg.begin % TILE == 0) return launch_lstage<S, RECON, EPI, CBC>(c, out, gauge, in, xin, e, parity, st, rg);
    }
    using A = typename Compute<S>::type;  // S is the storage type, A the arithmetic type
    const Epilogue<A> epi{(A)e.a, (A)e.g_re, (A)e.g_im, e.g5_out};
    // blocked map: all warps the register budget allows per SM in ONE block, on a compact box of warp tiles
    constexpr int NWARPS = MinBlocks<S, RECON>::value * 2;
    if constexpr (EPI == EPI_STORE)   // an experiment: only the plain dslash is instantiated with the blocked map
    if (c->kernel == LQCD_KERNEL_BLOCKED && rg.begin == 0 && rg.end == c->g.Vh && c->g.sz % TILE == 0) {
        BlockMap m = box_shape(NWARPS, c->g);
        const dim3 grid(m.gy * m.gz * ((c->g.T + m.bt - 1) / m.bt), parity < 0 ? 2 : 1);
        dslash_kernel<S, RECON, EPI, CBC, 32 * NWARPS><<<grid, 32 * NWARPS, 0, st>>>(
            (S*)out, (const S*)gauge, (const S*)in, (const S*)xin, epi, c->g, parity < 0 ? 0 : parity, make_bc<A>(c), rg.begin, rg.end, m);
        return after_launch();
    }
    constexpr int BLOCK = DSLASH_BLOCK;
    const dim3 grid((rg.end - rg.begin + BLOCK - 1) / BLOCK, parity < 0 ? 2 : 1);
    dslash_kernel<S, RECON, EPI, CBC, BLOCK><<<grid, BLOCK, 0, st>>>(
        (S*)out, (const S*)gauge, (const S*)in, (const S*)xin, epi, c->g, parity < 0 ? 0 : parity, make_bc<A>(c), rg.begin, rg.end, BlockMap{0, 0, 0, 0, 0, 0});
    return after_launch();
}

template <typename S, int RECON, int EPI>
lqcd_status launch_epi(const lqcd_ctx* c, void* out, const void* gauge, const void* in, const void* xin,
                       const EpiArgs& e, int parity, cudaStream_t st, CbRange rg) {
    return c->complex_bc ? launch_one<S, RECON, EPI, true>(c, out, gauge, in, xin, e, parity, st, rg)
                         : launch_one<S, RECON, EPI, false>(c, out, gauge, in, xin, e, parity, st, rg);
}

// out_p = epilogue(H in) for one storage type and link format; parity < 0: both parities, full fields.
// Explicitly instantiated in inst_*.cu.
template <typename S, int RECON>
lqcd_status launch_recon(const lqcd_ctx* c, void* out, const void* gauge, const void* in, const void* xin,
                         const EpiArgs& e, int parity, cudaStream_t st, CbRange rg) {
    switch (e.mode) {
        case EPI_STORE: return launch_epi<S, RECON, EPI_STORE>(c, out, gauge, in, xin, e, parity, st, rg);
        case EPI_XPAY: return launch_epi<S, RECON, EPI_XPAY>(c, out, gauge, in, xin, e, parity, st, rg);
        case EPI_G5SCALE: return launch_epi<S, RECON, EPI_G5SCALE>(c, out, gauge, in, xin, e, parity, st, rg);
        case EPI_G5XPAY: return launch_epi<S, RECON, EPI_G5XPAY>(c, out, gauge, in, xin, e, parity, st, rg);
    }
    return LQCD_EUNSUPPORTED;
}

#define LQCD_LAUNCH_RECON_ARGS \
    const lqcd_ctx*, void*, const void*, const void*, const void*, const EpiArgs&, int, cudaStream_t, CbRange

}  // namespace lqcd
