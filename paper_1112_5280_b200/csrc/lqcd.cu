// lqcd.cu -- host side of the C ABI declared in include/lqcd.h: argument checks, template
// dispatch (storage precision x recon x epilogue x bc kind x block size), kernel launches, the CG
// loops and the pipelined host-buffer path.  No field memory is allocated here; only the entry points
// that return results to host memory (lqcd_dslash_eo_host*, lqcd_cg_solve_tm*) synchronise.
#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <new>
#include <type_traits>

#include "blas_kernels.cuh"
#include "heatbath_kernels.cuh"
#include "pack_kernels.cuh"
#include "slab_launch.cuh"

using namespace lqcd;

namespace lqcd {
// the dslash kernels are instantiated in inst_*.cu
extern template lqcd_status launch_recon<double, 12>(LQCD_LAUNCH_RECON_ARGS);
extern template lqcd_status launch_recon<double, 18>(LQCD_LAUNCH_RECON_ARGS);
extern template lqcd_status launch_recon<float, 12>(LQCD_LAUNCH_RECON_ARGS);
extern template lqcd_status launch_recon<float, 18>(LQCD_LAUNCH_RECON_ARGS);
extern template lqcd_status launch_recon<__half, 12>(LQCD_LAUNCH_RECON_ARGS);
extern template lqcd_status launch_recon<float, RECON_12H>(LQCD_LAUNCH_RECON_ARGS);
extern template lqcd_status launch_recon<double, 8>(LQCD_LAUNCH_RECON_ARGS);
extern template lqcd_status launch_recon<float, 8>(LQCD_LAUNCH_RECON_ARGS);
extern template lqcd_status launch_slab<float>(LQCD_LAUNCH_SLAB_ARGS);
extern template lqcd_status launch_slab<double>(LQCD_LAUNCH_SLAB_ARGS);
extern template lqcd_status launch_push_faces<float>(LQCD_LAUNCH_FACES_ARGS);
extern template lqcd_status launch_push_faces<double>(LQCD_LAUNCH_FACES_ARGS);
}  // namespace lqcd

namespace {

std::atomic<unsigned long long> g_launches{0};
thread_local char g_cuda_err[256] = "";

lqcd_status cuda_fail(cudaError_t e) {
    std::strncpy(g_cuda_err, cudaGetErrorString(e), sizeof(g_cuda_err) - 1);
    return LQCD_ECUDA;
}

}  // namespace

lqcd_status lqcd::after_launch() {
    g_launches.fetch_add(1, std::memory_order_relaxed);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? LQCD_OK : cuda_fail(e);
}

namespace {

// Native fields are read and written with 256-bit words (fields.cuh): 32-byte alignment.  Canonical
// (interchange) buffers are only touched element by element by the pack kernels: the natural 16 bytes of a complex128.
inline bool aligned32(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 31u) == 0; }
inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

inline bool overlaps(const void* a, size_t na, const void* b, size_t nb) {
    const uintptr_t a0 = reinterpret_cast<uintptr_t>(a), b0 = reinterpret_cast<uintptr_t>(b);
    return a0 < b0 + nb && b0 < a0 + na;
}

inline size_t elem(const lqcd_ctx* c) { return c->p.precision / 8; }                      // stored element
inline size_t canon_elem(const lqcd_ctx* c) { return c->p.precision == 64 ? 8 : 4; }       // canonical element (16-bit storage: float)
// native half spinor, padded to whole tiles; 16-bit storage adds one fp32 norm per site
inline size_t half_bytes(const lqcd_ctx* c) {
    return (size_t)TILE * c->g.ntiles * (24 * elem(c) + (c->p.precision == 16 ? 4 : 0));
}
inline size_t align256(size_t n) { return (n + 255) & ~(size_t)255; }
constexpr int HOST_SLOTS = lqcd_host_pipe::SLOTS;  // pipeline depth of lqcd_dslash_eo_host_batch

inline CbRange all_sites(const lqcd_ctx* c) { return CbRange{0, c->g.Vh}; }

// out_p = epilogue(H in); parity < 0: both parities, full fields.
lqcd_status launch_dslash(const lqcd_ctx* c, void* out, const void* gauge, const void* in, const void* xin,
                          const EpiArgs& e, int parity, cudaStream_t st, CbRange rg) {
    if (c->p.precision == 16) return launch_recon<__half, 12>(c, out, gauge, in, xin, e, parity, st, rg);
    if (c->p.precision == 32) {
        if (c->p.link_precision == 16) return launch_recon<float, RECON_12H>(c, out, gauge, in, xin, e, parity, st, rg);
        if (c->p.recon == 8) return launch_recon<float, 8>(c, out, gauge, in, xin, e, parity, st, rg);
        return c->p.recon == 12 ? launch_recon<float, 12>(c, out, gauge, in, xin, e, parity, st, rg)
                                : launch_recon<float, 18>(c, out, gauge, in, xin, e, parity, st, rg);
    }
    if (c->p.recon == 8) return launch_recon<double, 8>(c, out, gauge, in, xin, e, parity, st, rg);
    return c->p.recon == 12 ? launch_recon<double, 12>(c, out, gauge, in, xin, e, parity, st, rg)
                            : launch_recon<double, 18>(c, out, gauge, in, xin, e, parity, st, rg);
}

lqcd_status check_fields(const lqcd_ctx* c, const void* out, const void* gauge, const void* in, size_t nbytes) {
    if (!c || !out || !gauge || !in) return LQCD_EINVAL;
    if (!aligned32(out) || !aligned32(gauge) || !aligned32(in)) return LQCD_EALIGN;
    if (overlaps(out, nbytes, in, nbytes)) return LQCD_EALIAS;
    return LQCD_OK;
}

}  // namespace

extern "C" {

lqcd_status lqcd_create(lqcd_ctx** ctx, const lqcd_params* p) {
    if (!ctx || !p) return LQCD_EINVAL;
    if (p->precision != 16 && p->precision != 32 && p->precision != 64) return LQCD_EINVAL;
    if (p->recon != 8 && p->recon != 12 && p->recon != 18) return LQCD_EINVAL;
    if (p->precision == 16 && p->recon != 12) return LQCD_EUNSUPPORTED;  // 16-bit storage: 12-real links only
    if (p->link_precision != 0 && p->link_precision != 16 && p->link_precision != p->precision) return LQCD_EINVAL;
    if (p->link_precision == 16 && (p->precision == 64 || p->recon != 12)) return LQCD_EUNSUPPORTED;
    if (p->recon == 8 && p->precision == 16) return LQCD_EUNSUPPORTED;  // 8-real links: fp32 / fp64 storage only
    double vol = 1;
    bool cbc = false;
    for (int mu = 0; mu < 4; ++mu) {
        if (p->dims[mu] < 4 || (p->dims[mu] & 1)) return LQCD_EINVAL;
        vol *= p->dims[mu];
        const double n2 = p->bc_re[mu] * p->bc_re[mu] + p->bc_im[mu] * p->bc_im[mu];
        if (!(std::fabs(n2 - 1.0) <= 1e-12)) return LQCD_EINVAL;
        if (p->bc_im[mu] != 0.0) cbc = true;
    }
    // checkerboard indices and in-tile word offsets are 32-bit; field offsets are size_t
    if (vol / 2 >= 1073741824.0) return LQCD_EUNSUPPORTED;
    lqcd_ctx* c = new (std::nothrow) lqcd_ctx;
    if (!c) return LQCD_EINVAL;
    c->p = *p;
    Geom& g = c->g;
    g.X = p->dims[0]; g.Y = p->dims[1]; g.Z = p->dims[2]; g.T = p->dims[3];
    g.Xh = g.X / 2;
    g.Vh = g.Xh * g.Y * g.Z * g.T;
    g.ntiles = (g.Vh + TILE - 1) / TILE;
    g.sy = g.Xh; g.sz = g.Xh * g.Y; g.st = g.Xh * g.Y * g.Z;
    g.tcf = g.T - 1; g.tcb = 0;
    set_fastdiv((unsigned)g.Xh, g.mul_xh, g.sh_xh);
    set_fastdiv((unsigned)g.Y, g.mul_y, g.sh_y);
    set_fastdiv((unsigned)g.Z, g.mul_z, g.sh_z);
    c->complex_bc = cbc;
    c->kernel = LQCD_KERNEL_GATHER;
    *ctx = c;
    return LQCD_OK;
}

lqcd_status lqcd_destroy(lqcd_ctx* ctx) {
    if (ctx && ctx->host.ready) {
        lqcd_host_pipe& h = ctx->host;
        for (int k = 0; k < lqcd_host_pipe::SLOTS; ++k) {
            cudaEventDestroy(h.in_done[k]);
            cudaEventDestroy(h.comp_done[k]);
            cudaEventDestroy(h.out_done[k]);
        }
        cudaEventDestroy(h.start);
        cudaStreamDestroy(h.up);
        cudaStreamDestroy(h.down);
    }
    delete ctx;
    return LQCD_OK;
}

size_t lqcd_spinor_bytes(const lqcd_ctx* c, int half) { return c ? half_bytes(c) * (half ? 1 : 2) : 0; }
size_t lqcd_gauge_bytes(const lqcd_ctx* c) {
    const size_t link_elem = c && c->p.link_precision == 16 ? 2 : (c ? elem(c) : 0);
    return c ? (size_t)2 * 8 * c->p.recon * TILE * c->g.ntiles * link_elem : 0;  // [parity][tile][hop 8][recon reals][32]
}
size_t lqcd_workspace_bytes(const lqcd_ctx* c) { return c ? half_bytes(c) : 0; }

size_t lqcd_host_workspace_bytes(const lqcd_ctx* c) {
    if (!c) return 0;
    const size_t canon_gauge = (size_t)4 * 2 * c->g.Vh * 18 * canon_elem(c);
    // per slot: canonical in, native in, native out, canonical out (the canonical half spinor is the larger one
    // with 16-bit storage)
    const size_t canon_half = (size_t)24 * c->g.Vh * canon_elem(c);
    return align256(lqcd_gauge_bytes(c)) + align256(canon_gauge) +
           HOST_SLOTS * 2 * (align256(half_bytes(c)) + align256(canon_half));
}

// 8-real links: the pack kernel raises this flag for a link the decoder cannot rebuild.  One flag per GPU, inside the
// library image (the library allocates nothing); g_recon8_lock keeps the clear / launch / read-back of two packs apart.
static __device__ unsigned g_recon8_bad;
static std::mutex g_recon8_lock;

// Smallest admissible min(|U00|, sqrt(|U01|^2 + |U02|^2), |U20|) of a link stored with 8 reals: the decoder loses digits
// like eps / margin, so below 64 eps not even two digits of the rebuilt rows are right (0: unit links, NaN).
static double recon8_min_margin(int precision) { return 64.0 * (precision == 64 ? 0x1p-53 : 0x1p-24); }

static lqcd_status pack_gauge8_checked(const lqcd_ctx* c, void* native, const void* canon, const void* below, dim3 grid,
                                       cudaStream_t st) {
    std::lock_guard<std::mutex> guard(g_recon8_lock);
    unsigned* bad_dev = nullptr;
    unsigned bad = 0;
    cudaError_t e;
    if ((e = cudaGetSymbolAddress((void**)&bad_dev, g_recon8_bad)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaMemsetAsync(bad_dev, 0, sizeof(unsigned), st)) != cudaSuccess) return cuda_fail(e);
    const double m = recon8_min_margin(c->p.precision);
    if (c->p.precision == 32) pack_gauge8_kernel<float><<<grid, 128, 0, st>>>((float*)native, (const float*)canon, (const float*)below, c->g, m * m, bad_dev);
    else pack_gauge8_kernel<double><<<grid, 128, 0, st>>>((double*)native, (const double*)canon, (const double*)below, c->g, m * m, bad_dev);
    lqcd_status s = after_launch();
    if (s != LQCD_OK) return s;
    if ((e = cudaMemcpyAsync(&bad, bad_dev, sizeof(unsigned), cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e);
    return bad ? LQCD_EUNSUPPORTED : LQCD_OK;   // the field has a link outside the 8-real encoding: store it with 12
}

static lqcd_status pack_gauge_impl(const lqcd_ctx* c, void* native, const void* canon, const void* below, void* stream) {
    if (!c || !native || !canon) return LQCD_EINVAL;
    if (!aligned32(native) || !aligned16(canon) || !aligned16(below)) return LQCD_EALIGN;
    const dim3 grid((c->g.Vh + 127) / 128, 8, 2);
    cudaStream_t st = (cudaStream_t)stream;
    if (c->p.precision == 16 || c->p.link_precision == 16) {
        pack_gauge_h_kernel<<<grid, 128, 0, st>>>((__half*)native, (const float*)canon, (const float*)below, c->g);
    } else if (c->p.recon == 8) {
        return pack_gauge8_checked(c, native, canon, below, grid, st);
    } else if (c->p.precision == 32) {
        if (c->p.recon == 12) pack_gauge_kernel<float, 12><<<grid, 128, 0, st>>>((float*)native, (const float*)canon, (const float*)below, c->g);
        else pack_gauge_kernel<float, 18><<<grid, 128, 0, st>>>((float*)native, (const float*)canon, (const float*)below, c->g);
    } else {
        if (c->p.recon == 12) pack_gauge_kernel<double, 12><<<grid, 128, 0, st>>>((double*)native, (const double*)canon, (const double*)below, c->g);
        else pack_gauge_kernel<double, 18><<<grid, 128, 0, st>>>((double*)native, (const double*)canon, (const double*)below, c->g);
    }
    return after_launch();
}

lqcd_status lqcd_pack_gauge(const lqcd_ctx* c, void* native, const void* canon, void* stream) {
    return pack_gauge_impl(c, native, canon, nullptr, stream);
}

lqcd_status lqcd_pack_gauge_slab(const lqcd_ctx* c, void* native, const void* canon, const void* tlinks_below, void* stream) {
    if (!tlinks_below) return LQCD_EINVAL;
    return pack_gauge_impl(c, native, canon, tlinks_below, stream);
}

lqcd_status lqcd_gauge_recon8_margin(const lqcd_ctx* c, const void* canon, void* scratch, double* margin_host, void* stream) {
    if (!c || !canon || !scratch || !margin_host) return LQCD_EINVAL;
    if (c->p.precision == 16) return LQCD_EUNSUPPORTED;
    if (!aligned16(canon) || (reinterpret_cast<uintptr_t>(scratch) & 7u)) return LQCD_EALIGN;
    cudaStream_t st = (cudaStream_t)stream;
    const double one = 1.0;
    cudaError_t e;
    if ((e = cudaMemcpyAsync(scratch, &one, sizeof(one), cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_fail(e);
    const size_t nlinks = (size_t)8 * c->g.Vh;
    const unsigned grid = (unsigned)((nlinks + 255) / 256);
    if (c->p.precision == 64) recon8_margin_kernel<double><<<grid, 256, 0, st>>>((const double*)canon, nlinks, (unsigned long long*)scratch);
    else recon8_margin_kernel<float><<<grid, 256, 0, st>>>((const float*)canon, nlinks, (unsigned long long*)scratch);
    lqcd_status s = after_launch();
    if (s != LQCD_OK) return s;
    double m2 = 0.0;
    if ((e = cudaMemcpyAsync(&m2, scratch, sizeof(m2), cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e);
    *margin_host = std::sqrt(m2);
    return LQCD_OK;
}

static lqcd_status pack_unpack(const lqcd_ctx* c, void* dst, const void* src, int parity, void* stream, bool unpack) {
    if (!c || !dst || !src) return LQCD_EINVAL;
    if (parity < -1 || parity > 1) return LQCD_EINVAL;
    if (!aligned32(unpack ? src : dst) || !aligned16(unpack ? dst : src)) return LQCD_EALIGN;  // native 32, canonical 16
    const dim3 grid((c->g.Vh + 127) / 128, parity < 0 ? 2 : 1);
    cudaStream_t st = (cudaStream_t)stream;
    if (c->p.precision == 16) {
        if (unpack) pack_spinor_h_kernel<true><<<grid, 128, 0, st>>>(dst, src, c->g, parity);
        else pack_spinor_h_kernel<false><<<grid, 128, 0, st>>>(dst, src, c->g, parity);
    } else if (c->p.precision == 32) {
        if (unpack) pack_spinor_kernel<float, true><<<grid, 128, 0, st>>>((float*)dst, (const float*)src, c->g, parity);
        else pack_spinor_kernel<float, false><<<grid, 128, 0, st>>>((float*)dst, (const float*)src, c->g, parity);
    } else {
        if (unpack) pack_spinor_kernel<double, true><<<grid, 128, 0, st>>>((double*)dst, (const double*)src, c->g, parity);
        else pack_spinor_kernel<double, false><<<grid, 128, 0, st>>>((double*)dst, (const double*)src, c->g, parity);
    }
    return after_launch();
}

lqcd_status lqcd_pack_spinor(const lqcd_ctx* c, void* native, const void* canon, int parity, void* stream) {
    return pack_unpack(c, native, canon, parity, stream, false);
}

lqcd_status lqcd_unpack_spinor(const lqcd_ctx* c, void* canon, const void* native, int parity, void* stream) {
    return pack_unpack(c, canon, native, parity, stream, true);
}

lqcd_status lqcd_set_kernel(lqcd_ctx* c, int kernel) {
    if (!c || kernel < LQCD_KERNEL_GATHER || kernel > LQCD_KERNEL_LSTAGE) return LQCD_EINVAL;
    if ((kernel == LQCD_KERNEL_PIPE || kernel == LQCD_KERNEL_LSTAGE) && (c->p.precision == 16 || c->p.link_precision == 16)) return LQCD_EUNSUPPORTED;
    c->kernel = kernel;
    return LQCD_OK;
}

lqcd_status lqcd_dslash_full(const lqcd_ctx* c, void* out, const void* gauge, const void* in, void* stream) {
    lqcd_status s = check_fields(c, out, gauge, in, c ? 2 * half_bytes(c) : 0);
    if (s != LQCD_OK) return s;
    return launch_dslash(c, out, gauge, in, nullptr, EpiArgs{EPI_STORE, 0, 0, 0, 0}, -1, (cudaStream_t)stream, all_sites(c));
}

lqcd_status lqcd_dslash_eo(const lqcd_ctx* c, void* out, const void* gauge, const void* in, int out_parity,
                           void* stream) {
    if (out_parity != 0 && out_parity != 1) return LQCD_EINVAL;
    lqcd_status s = check_fields(c, out, gauge, in, c ? half_bytes(c) : 0);
    if (s != LQCD_OK) return s;
    return launch_dslash(c, out, gauge, in, nullptr, EpiArgs{EPI_STORE, 0, 0, 0, 0}, out_parity, (cudaStream_t)stream, all_sites(c));
}

// ---- next row f3: time-slab decomposition (slab_kernels.cuh) ----------------------------------------------
// A rank of a T-slab decomposition holds the time slices [t0, t0 + T_loc) of the global lattice (T_loc even) as a
// local lattice of exactly those slices.  The t hops that leave the slab read projected half spinors from two halo
// buffers filled by the neighbouring ranks (lqcd_slab_push_faces); the interior slices need no halo and are plain
// lqcd_dslash_eo_range launches.  The boundary phase sits where the global boundary cuts the slab, not at the local wrap.
lqcd_status lqcd_set_time_slab(lqcd_ctx* c, int t_cross_fwd, int t_cross_bwd) {
    if (!c) return LQCD_EINVAL;
    if (t_cross_fwd < -1 || t_cross_fwd >= c->g.T || t_cross_bwd < -1 || t_cross_bwd >= c->g.T) return LQCD_EINVAL;
    c->g.tcf = t_cross_fwd;
    c->g.tcb = t_cross_bwd;
    return LQCD_OK;
}

lqcd_status lqcd_dslash_eo_range(const lqcd_ctx* c, void* out, const void* gauge, const void* in, int out_parity,
                                 int t_begin, int t_end, void* stream) {
    if (out_parity != 0 && out_parity != 1) return LQCD_EINVAL;
    lqcd_status s = check_fields(c, out, gauge, in, c ? half_bytes(c) : 0);
    if (s != LQCD_OK) return s;
    if (t_begin < 0 || t_end > c->g.T || t_begin > t_end) return LQCD_EINVAL;
    if (t_begin == t_end) return LQCD_OK;
    return launch_dslash(c, out, gauge, in, nullptr, EpiArgs{EPI_STORE, 0, 0, 0, 0}, out_parity, (cudaStream_t)stream,
                         CbRange{t_begin * c->g.st, t_end * c->g.st});
}

static bool slab_capable(const lqcd_ctx* c) { return c->p.precision != 16 && c->p.link_precision != 16; }

size_t lqcd_halo_bytes(const lqcd_ctx* c) {
    // one face of projected half spinors: 12 reals per site of one parity of a time slice, padded to whole 32-site tiles
    if (!c || !slab_capable(c)) return 0;
    return (size_t)face_tiles(c->g) * TILE * 12 * elem(c);
}

lqcd_status lqcd_slab_push_faces(const lqcd_ctx* c, const void* in, void* dst_up, void* dst_down, void* flag_up, void* flag_down,
                                 unsigned long long epoch, void* stream) {
    if (!c || !in) return LQCD_EINVAL;
    if (!slab_capable(c)) return LQCD_EUNSUPPORTED;
    if (!aligned32(in) || !aligned32(dst_up) || !aligned32(dst_down)) return LQCD_EALIGN;
    if ((reinterpret_cast<uintptr_t>(flag_up) | reinterpret_cast<uintptr_t>(flag_down)) & 7u) return LQCD_EALIGN;
    if (!dst_up && !dst_down) return LQCD_OK;
    return c->p.precision == 32
               ? launch_push_faces<float>(c, in, dst_up, dst_down, (unsigned long long*)flag_up, (unsigned long long*)flag_down, epoch, (cudaStream_t)stream)
               : launch_push_faces<double>(c, in, dst_up, dst_down, (unsigned long long*)flag_up, (unsigned long long*)flag_down, epoch, (cudaStream_t)stream);
}

lqcd_status lqcd_dslash_eo_slab(const lqcd_ctx* c, void* out, const void* gauge, const void* in, const void* halo_from_up,
                                const void* halo_from_down, const void* wait_up, const void* wait_down, unsigned long long epoch,
                                int out_parity, int t_begin, int t_end, void* stream) {
    if (out_parity != 0 && out_parity != 1) return LQCD_EINVAL;
    lqcd_status s = check_fields(c, out, gauge, in, c ? half_bytes(c) : 0);
    if (s != LQCD_OK) return s;
    if (!slab_capable(c)) return LQCD_EUNSUPPORTED;
    if (!halo_from_up || !halo_from_down) return LQCD_EINVAL;
    if (!aligned32(halo_from_up) || !aligned32(halo_from_down)) return LQCD_EALIGN;
    if ((reinterpret_cast<uintptr_t>(wait_up) | reinterpret_cast<uintptr_t>(wait_down)) & 7u) return LQCD_EALIGN;
    if (t_begin < 0 || t_end > c->g.T || t_begin > t_end) return LQCD_EINVAL;
    if (t_begin == t_end) return LQCD_OK;
    const CbRange rg{t_begin * c->g.st, t_end * c->g.st};
    return c->p.precision == 32
               ? launch_slab<float>(c, out, gauge, in, halo_from_up, halo_from_down, (const unsigned long long*)wait_up,
                                    (const unsigned long long*)wait_down, epoch, out_parity, (cudaStream_t)stream, rg)
               : launch_slab<double>(c, out, gauge, in, halo_from_up, halo_from_down, (const unsigned long long*)wait_up,
                                     (const unsigned long long*)wait_down, epoch, out_parity, (cudaStream_t)stream, rg);
}

// Shared body of lqcd_apply_M (theta = 0) and lqcd_apply_M_tm (theta = 2 kappa mu).
static lqcd_status apply_M_impl(const lqcd_ctx* c, void* out, const void* gauge, const void* in, double kappa,
                                double theta, bool twisted, int eo, void* workspace, cudaStream_t st, int g5_out = 0) {
    if (eo != 0 && eo != 1) return LQCD_EINVAL;
    const EpiArgs last{twisted ? EPI_G5XPAY : EPI_XPAY, eo ? -kappa * kappa : -kappa, 1.0, theta, g5_out};
    if (eo == 0) {
        lqcd_status s = check_fields(c, out, gauge, in, c ? 2 * half_bytes(c) : 0);
        if (s != LQCD_OK) return s;
        return launch_dslash(c, out, gauge, in, in, last, -1, st, all_sites(c));  // out = (1 + i theta g5) in - kappa H in
    }
    const size_t hb = c ? half_bytes(c) : 0;
    lqcd_status s = check_fields(c, out, gauge, in, hb);
    if (s != LQCD_OK) return s;
    if (!workspace) return LQCD_EINVAL;
    if (!aligned32(workspace)) return LQCD_EALIGN;
    if (overlaps(workspace, hb, in, hb) || overlaps(workspace, hb, out, hb)) return LQCD_EALIAS;
    // tmp_o = (1 + i theta g5)^-1 H_oe in_e, with (1 + i theta g5)^-1 = (1 - i theta g5) / (1 + theta^2)
    const double n = 1.0 / (1.0 + theta * theta);
    const EpiArgs first{twisted ? EPI_G5SCALE : EPI_STORE, 0.0, n, -theta * n, 0};
    s = launch_dslash(c, workspace, gauge, in, nullptr, first, 1, st, all_sites(c));
    if (s != LQCD_OK) return s;
    return launch_dslash(c, out, gauge, workspace, in, last, 0, st, all_sites(c));  // out_e = (1 + i theta g5) in_e - kappa^2 H_eo tmp_o
}

lqcd_status lqcd_apply_M(const lqcd_ctx* c, void* out, const void* gauge, const void* in, double kappa, int eo,
                         void* workspace, void* stream) {
    return apply_M_impl(c, out, gauge, in, kappa, 0.0, false, eo, workspace, (cudaStream_t)stream);
}

lqcd_status lqcd_apply_M_tm(const lqcd_ctx* c, void* out, const void* gauge, const void* in, double kappa, double mu,
                            int eo, void* workspace, void* stream) {
    return apply_M_impl(c, out, gauge, in, kappa, 2.0 * kappa * mu, true, eo, workspace, (cudaStream_t)stream);
}

// ---- next row f2: CG on the normal equations of the even-odd twisted-mass matrix -------------------------
// A = Mhat(mu)^+ Mhat(mu) = Q(-mu) Q(mu) with Q(mu) = gamma_5 Mhat(mu)  (gamma_5 Mhat(mu) gamma_5 = Mhat(-mu)^+).

}  // extern "C" (templates below)

namespace {

struct CgWorkspace {
    char *r, *p, *t, *s, *tmp;
    double* partial;
    CgScalars* sc;
    int nblk;
};

// native half spinor of precision `prec` on the lattice of c (bytes, padded to whole tiles)
inline size_t half_bytes_of(const lqcd_ctx* c, int prec) {
    return (size_t)TILE * c->g.ntiles * (prec == 16 ? 24 * 2 + 4 : 24 * (prec / 8));
}
// storage precision of the CG iterate and residual for an operator context: 16-bit operators iterate with fp32 x and r
inline int cg_x_precision(const lqcd_ctx* c) { return c->p.precision == 16 ? 32 : c->p.precision; }

// r in the iterate's format; p, t = Q p, s = A p and the operator's intermediate in the operator's format
CgWorkspace carve_cg(const lqcd_ctx* c, void* ws) {
    CgWorkspace w;
    const size_t hx = align256(half_bytes_of(c, cg_x_precision(c))), hp = align256(half_bytes(c));
    char* base = static_cast<char*>(ws);
    w.r = base; w.p = base + hx; w.t = w.p + hp; w.s = w.t + hp; w.tmp = w.s + hp;
    w.nblk = (c->g.Vh + BLAS_BLOCK - 1) / BLAS_BLOCK;
    w.partial = reinterpret_cast<double*>(w.tmp + hp);
    w.sc = reinterpret_cast<CgScalars*>(w.tmp + hp + align256((size_t)w.nblk * sizeof(double)));
    return w;
}

// X: storage type of x, b, r;  P: storage type of the operator context c (p, Q p, A p)
template <typename X, typename P>
lqcd_status cg_loop(const lqcd_ctx* c, void* x, const void* gauge, const void* b, double kappa, double mu, double tol,
                    int maxiter, const CgWorkspace& w, int* iters_out, double* relres_out, cudaStream_t st) {
    const size_t hx = half_bytes_of(c, cg_x_precision(c));
    const double theta = 2.0 * kappa * mu;
    const Geom& g = c->g;
    cudaError_t e;
    lqcd_status s;
    // x = 0, r = p = b, rr = bb = <b, b>
    CgScalars init{};
    init.tol2 = tol * tol;
    if ((e = cudaMemcpyAsync(w.sc, &init, sizeof(init), cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaMemsetAsync(x, 0, hx, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaMemcpyAsync(w.r, b, hx, cudaMemcpyDeviceToDevice, st)) != cudaSuccess) return cuda_fail(e);
    if constexpr (std::is_same<X, P>::value) {
        if ((e = cudaMemcpyAsync(w.p, b, hx, cudaMemcpyDeviceToDevice, st)) != cudaSuccess) return cuda_fail(e);
    } else {
        convert_kernel<P, X><<<w.nblk, BLAS_BLOCK, 0, st>>>((P*)w.p, (const X*)b, g);
        if ((s = after_launch()) != LQCD_OK) return s;
    }
    norm2_kernel<X><<<w.nblk, BLAS_BLOCK, 0, st>>>((const X*)b, g, w.partial);
    if ((s = after_launch()) != LQCD_OK) return s;
    cg_scalar_kernel<<<1, BLAS_BLOCK, 0, st>>>(w.partial, w.nblk, w.sc, CG_OP_INIT);
    if ((s = after_launch()) != LQCD_OK) return s;

    // Iterations enqueued between two looks at the convergence flag: 8 while the residual is far from the
    // target, 1 once |r|^2 is within a factor 1000 of it (so at most a few iterations are enqueued in vain).
    constexpr int CHECK_EVERY = 8;
    CgScalars host{};
    host.rr = host.bb = 1.0;
    for (int it = 0; it < maxiter;) {
        const int want = host.rr <= 1e3 * init.tol2 * host.bb ? 1 : CHECK_EVERY;
        const int chunk = (maxiter - it < want) ? maxiter - it : want;
        for (int k = 0; k < chunk; ++k) {
            // t = Q(mu) p ; alpha = rr / |t|^2
            if ((s = apply_M_impl(c, w.t, gauge, w.p, kappa, theta, true, 1, w.tmp, st, 1)) != LQCD_OK) return s;
            norm2_kernel<P><<<w.nblk, BLAS_BLOCK, 0, st>>>((const P*)w.t, g, w.partial);
            if ((s = after_launch()) != LQCD_OK) return s;
            cg_scalar_kernel<<<1, BLAS_BLOCK, 0, st>>>(w.partial, w.nblk, w.sc, CG_OP_PAP);
            if ((s = after_launch()) != LQCD_OK) return s;
            // s = Q(-mu) t = A p ; x += alpha p ; r -= alpha s ; rr', beta, convergence
            if ((s = apply_M_impl(c, w.s, gauge, w.t, kappa, -theta, true, 1, w.tmp, st, 1)) != LQCD_OK) return s;
            cg_update_xr_kernel<X, P><<<w.nblk, BLAS_BLOCK, 0, st>>>((X*)x, (X*)w.r, (const P*)w.p, (const P*)w.s, g, w.sc, w.partial);
            if ((s = after_launch()) != LQCD_OK) return s;
            cg_scalar_kernel<<<1, BLAS_BLOCK, 0, st>>>(w.partial, w.nblk, w.sc, CG_OP_RR);
            if ((s = after_launch()) != LQCD_OK) return s;
            cg_update_p_kernel<X, P><<<w.nblk, BLAS_BLOCK, 0, st>>>((P*)w.p, (const X*)w.r, g, w.sc);
            if ((s = after_launch()) != LQCD_OK) return s;
        }
        it += chunk;
        if ((e = cudaMemcpyAsync(&host, w.sc, sizeof(host), cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
        if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e);
        if (host.done) break;
    }
    if (!host.done) {
        if ((e = cudaMemcpyAsync(&host, w.sc, sizeof(host), cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
        if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e);
    }
    if (iters_out) *iters_out = host.iters;
    if (relres_out) *relres_out = host.bb > 0.0 ? std::sqrt(host.rr / host.bb) : 0.0;
    return LQCD_OK;
}

// |v|^2 of a native half spinor, to host (synchronises the stream)
template <typename R>
lqcd_status norm2_to_host(const lqcd_ctx* c, const void* v, double* partial, double* scratch, double* out, cudaStream_t st) {
    const int nblk = (c->g.Vh + BLAS_BLOCK - 1) / BLAS_BLOCK;
    lqcd_status s;
    norm2_kernel<R><<<nblk, BLAS_BLOCK, 0, st>>>((const R*)v, c->g, partial);
    if ((s = after_launch()) != LQCD_OK) return s;
    sum_partials_kernel<<<1, BLAS_BLOCK, 0, st>>>(partial, nblk, scratch);
    if ((s = after_launch()) != LQCD_OK) return s;
    cudaError_t e;
    if ((e = cudaMemcpyAsync(out, scratch, sizeof(double), cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e);
    return LQCD_OK;
}

}  // namespace

extern "C" {

// the loop's own scratch (carve_cg)
static size_t cg_loop_bytes(const lqcd_ctx* c) {
    const int nblk = (c->g.Vh + BLAS_BLOCK - 1) / BLAS_BLOCK;
    return align256(half_bytes_of(c, cg_x_precision(c))) + 4 * align256(half_bytes(c)) + align256((size_t)nblk * sizeof(double)) +
           align256(sizeof(CgScalars));
}

size_t lqcd_cg_workspace_bytes(const lqcd_ctx* c) {
    if (!c) return 0;
    // a 16-bit context iterates on fp32 copies of b and x: two more fp32 half spinors
    return cg_loop_bytes(c) + (c->p.precision == 16 ? 2 * align256(half_bytes_of(c, 32)) : 0);
}

lqcd_status lqcd_apply_Q_tm(const lqcd_ctx* c, void* out, const void* gauge, const void* in, double kappa, double mu,
                            void* workspace, void* stream) {
    return apply_M_impl(c, out, gauge, in, kappa, 2.0 * kappa * mu, true, 1, workspace, (cudaStream_t)stream, 1);
}

lqcd_status lqcd_cg_solve_tm(const lqcd_ctx* c, void* x, const void* gauge, const void* b, double kappa, double mu,
                             double tol, int maxiter, void* workspace, int* iters_out, double* relres_out, void* stream) {
    const size_t hb = c ? half_bytes(c) : 0;
    lqcd_status s = check_fields(c, x, gauge, b, hb);
    if (s != LQCD_OK) return s;
    if (!workspace || !(tol > 0.0) || maxiter < 0) return LQCD_EINVAL;
    if (reinterpret_cast<uintptr_t>(workspace) & 255u) return LQCD_EALIGN;
    const size_t wb = lqcd_cg_workspace_bytes(c);
    if (overlaps(workspace, wb, x, hb) || overlaps(workspace, wb, b, hb)) return LQCD_EALIAS;
    cudaStream_t st = (cudaStream_t)stream;
    if (c->p.precision == 16) {
        // 16-bit storage: the iterate and the residual live in fp32 (their recurrences carry the accuracy), the search
        // direction and the operator's vectors in the 16-bit format; b is widened first, x rounded to storage at the end
        char* b32 = static_cast<char*>(workspace);
        char* x32 = b32 + align256(half_bytes_of(c, 32));
        const CgWorkspace w = carve_cg(c, x32 + align256(half_bytes_of(c, 32)));
        convert_kernel<float, __half><<<w.nblk, BLAS_BLOCK, 0, st>>>((float*)b32, (const __half*)b, c->g);
        if ((s = after_launch()) != LQCD_OK) return s;
        s = cg_loop<float, __half>(c, x32, gauge, b32, kappa, mu, tol, maxiter, w, iters_out, relres_out, st);
        if (s != LQCD_OK) return s;
        convert_kernel<__half, float><<<w.nblk, BLAS_BLOCK, 0, st>>>((__half*)x, (const float*)x32, c->g);
        if ((s = after_launch()) != LQCD_OK) return s;
        const cudaError_t e = cudaStreamSynchronize(st);
        return e == cudaSuccess ? LQCD_OK : cuda_fail(e);
    }
    const CgWorkspace w = carve_cg(c, workspace);
    return c->p.precision == 32 ? cg_loop<float, float>(c, x, gauge, b, kappa, mu, tol, maxiter, w, iters_out, relres_out, st)
                                : cg_loop<double, double>(c, x, gauge, b, kappa, mu, tol, maxiter, w, iters_out, relres_out, st);
}

// Mixed precision: fp64 defect correction around the fp32 CG (reading F2).
//   x = 0, r = b;  repeat { solve A32 e = (float) r to inner_tol with lqcd_cg_solve_tm's loop;  x += e;
//   r = b - A64 x (true residual, fp64) } until |r| <= tol |b|.
size_t lqcd_cg_mixed_workspace_bytes(const lqcd_ctx* c64, const lqcd_ctx* c32) {
    if (!c64 || !c32) return 0;
    const int nblk = (c64->g.Vh + BLAS_BLOCK - 1) / BLAS_BLOCK;
    return 4 * align256(half_bytes(c64)) + 2 * align256(half_bytes_of(c32, 32)) + align256(cg_loop_bytes(c32)) +
           align256((size_t)nblk * sizeof(double)) + 256;
}

lqcd_status lqcd_cg_solve_tm_mixed(const lqcd_ctx* c64, const lqcd_ctx* c32, void* x, const void* gauge64,
                                   const void* gauge32, const void* b, double kappa, double mu, double tol,
                                   double inner_tol, int maxiter, void* workspace, int* iters_out, int* outer_out,
                                   double* relres_out, void* stream) {
    if (!c64 || !c32 || !gauge32) return LQCD_EINVAL;
    if (c64->p.precision != 64 || (c32->p.precision != 32 && c32->p.precision != 16)) return LQCD_EINVAL;
    for (int m = 0; m < 4; ++m)
        if (c64->p.dims[m] != c32->p.dims[m] || c64->p.bc_re[m] != c32->p.bc_re[m] || c64->p.bc_im[m] != c32->p.bc_im[m])
            return LQCD_EINVAL;
    const size_t hb64 = half_bytes(c64), hb32 = half_bytes_of(c32, 32);   // the inner iterate and residual are fp32 also for a 16-bit inner operator
    lqcd_status s = check_fields(c64, x, gauge64, b, hb64);
    if (s != LQCD_OK) return s;
    if (!workspace || !(tol > 0.0) || !(inner_tol > 0.0) || maxiter < 0) return LQCD_EINVAL;
    if (!aligned32(gauge32)) return LQCD_EALIGN;
    if (reinterpret_cast<uintptr_t>(workspace) & 255u) return LQCD_EALIGN;
    const size_t wb = lqcd_cg_mixed_workspace_bytes(c64, c32);
    if (overlaps(workspace, wb, x, hb64) || overlaps(workspace, wb, b, hb64)) return LQCD_EALIAS;

    cudaStream_t st = (cudaStream_t)stream;
    const Geom& g = c64->g;
    const int nblk = (g.Vh + BLAS_BLOCK - 1) / BLAS_BLOCK;
    char* base = static_cast<char*>(workspace);
    char* r64 = base;                   base += align256(hb64);
    char* s64 = base;                   base += align256(hb64);
    char* t64 = base;                   base += align256(hb64);
    char* tmp64 = base;                 base += align256(hb64);
    char* r32 = base;                   base += align256(hb32);
    char* e32 = base;                   base += align256(hb32);
    char* inner_ws = base;              base += align256(cg_loop_bytes(c32));
    double* partial = reinterpret_cast<double*>(base);  base += align256((size_t)nblk * sizeof(double));
    double* scratch = reinterpret_cast<double*>(base);
    const CgWorkspace iw = carve_cg(c32, inner_ws);
    const double theta = 2.0 * kappa * mu;

    cudaError_t e;
    double bb = 0.0, rr = 0.0;
    if ((s = norm2_to_host<double>(c64, b, partial, scratch, &bb, st)) != LQCD_OK) return s;
    if ((e = cudaMemsetAsync(x, 0, hb64, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaMemcpyAsync(r64, b, hb64, cudaMemcpyDeviceToDevice, st)) != cudaSuccess) return cuda_fail(e);
    rr = bb;
    int total = 0, outer = 0;
    while (bb > 0.0 && rr > tol * tol * bb && total < maxiter && outer < 50) {
        // inner solve in fp32: A e = r, relative tolerance inner_tol but never tighter than what is still needed
        convert_kernel<float, double><<<nblk, BLAS_BLOCK, 0, st>>>((float*)r32, (const double*)r64, g);
        if ((s = after_launch()) != LQCD_OK) return s;
        const double need = tol * std::sqrt(bb / rr);  // relative reduction of |r| still required
        int it = 0;
        const double itol = inner_tol > 0.5 * need ? inner_tol : 0.5 * need;
        s = c32->p.precision == 16 ? cg_loop<float, __half>(c32, e32, gauge32, r32, kappa, mu, itol, maxiter - total, iw, &it, nullptr, st)
                                   : cg_loop<float, float>(c32, e32, gauge32, r32, kappa, mu, itol, maxiter - total, iw, &it, nullptr, st);
        if (s != LQCD_OK) return s;
        total += it;
        ++outer;
        // x += e;  r = b - A x in fp64
        accumulate_correction_kernel<<<nblk, BLAS_BLOCK, 0, st>>>((double*)x, (const float*)e32, g);
        if ((s = after_launch()) != LQCD_OK) return s;
        if ((s = apply_M_impl(c64, t64, gauge64, x, kappa, theta, true, 1, tmp64, st, 1)) != LQCD_OK) return s;
        if ((s = apply_M_impl(c64, s64, gauge64, t64, kappa, -theta, true, 1, tmp64, st, 1)) != LQCD_OK) return s;
        residual_kernel<double><<<nblk, BLAS_BLOCK, 0, st>>>((double*)r64, (const double*)b, (const double*)s64, g, partial);
        if ((s = after_launch()) != LQCD_OK) return s;
        sum_partials_kernel<<<1, BLAS_BLOCK, 0, st>>>(partial, nblk, scratch);
        if ((s = after_launch()) != LQCD_OK) return s;
        const double rr_old = rr;
        if ((e = cudaMemcpyAsync(&rr, scratch, sizeof(double), cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
        if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e);
        if (it == 0 || !(rr < rr_old)) break;  // no progress: fp32 cannot reduce this residual further
    }
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e);
    if (iters_out) *iters_out = total;
    if (outer_out) *outer_out = outer;
    if (relres_out) *relres_out = bb > 0.0 ? std::sqrt(rr / bb) : 0.0;
    return LQCD_OK;
}

// Host-buffer path.  Items are pipelined over HOST_SLOTS device slots and three streams (upload, the caller's
// stream for the kernels, download), so the two PCIe directions and the kernels overlap.
lqcd_status lqcd_dslash_eo_host_batch(const lqcd_ctx* c, int n, void* const* out_host, const void* gauge_host,
                                      const void* const* in_host, const int* out_parity, void* ws, void* stream) {
    if (!c || n < 0 || (n > 0 && (!out_host || !in_host || !out_parity)) || !ws) return LQCD_EINVAL;
    for (int i = 0; i < n; ++i)
        if (!out_host[i] || !in_host[i] || (out_parity[i] != 0 && out_parity[i] != 1)) return LQCD_EINVAL;
    if (reinterpret_cast<uintptr_t>(ws) & 255u) return LQCD_EALIGN;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t hb = half_bytes(c);                             // native half spinor (padded to whole tiles)
    const size_t cb_bytes = (size_t)24 * c->g.Vh * canon_elem(c);     // canonical half spinor
    const size_t canon_gauge = (size_t)4 * 2 * c->g.Vh * 18 * canon_elem(c);
    char* base = static_cast<char*>(ws);
    char* g_nat = base;                 base += align256(lqcd_gauge_bytes(c));
    char* g_can = base;                 base += align256(canon_gauge);
    char *in_can[HOST_SLOTS], *in_nat[HOST_SLOTS], *out_nat[HOST_SLOTS], *out_can[HOST_SLOTS];
    for (int k = 0; k < HOST_SLOTS; ++k) {
        in_can[k] = base;  base += align256(cb_bytes);
        in_nat[k] = base;  base += align256(hb);
        out_nat[k] = base; base += align256(hb);
        out_can[k] = base; base += align256(cb_bytes);
    }
    cudaError_t e = cudaSuccess;
    lqcd_status s = LQCD_OK;
    auto fail = [&](cudaError_t err) { e = err; return err != cudaSuccess; };
    lqcd_host_pipe& hp = c->host;
    std::lock_guard<std::mutex> guard(hp.lock);
    if (!hp.ready) {   // first host-path call on this context: two copy streams and the events that order the slots
        bool ok = !fail(cudaStreamCreateWithFlags(&hp.up, cudaStreamNonBlocking)) &&
                  !fail(cudaStreamCreateWithFlags(&hp.down, cudaStreamNonBlocking)) &&
                  !fail(cudaEventCreateWithFlags(&hp.start, cudaEventDisableTiming));
        for (int k = 0; k < HOST_SLOTS && ok; ++k)
            ok = !fail(cudaEventCreateWithFlags(&hp.in_done[k], cudaEventDisableTiming)) &&
                 !fail(cudaEventCreateWithFlags(&hp.comp_done[k], cudaEventDisableTiming)) &&
                 !fail(cudaEventCreateWithFlags(&hp.out_done[k], cudaEventDisableTiming));
        if (!ok) return cuda_fail(e);   // a context whose host path could not be set up keeps failing here
        hp.ready = true;
    }
    const cudaStream_t up = hp.up, down = hp.down;
    const cudaEvent_t start = hp.start;
    cudaEvent_t* const in_done = hp.in_done;
    cudaEvent_t* const comp_done = hp.comp_done;
    cudaEvent_t* const out_done = hp.out_done;
    do {
        // everything already enqueued on the caller's stream comes first
        if (fail(cudaEventRecord(start, st)) || fail(cudaStreamWaitEvent(up, start, 0)) || fail(cudaStreamWaitEvent(down, start, 0))) break;
        if (gauge_host) {
            if (fail(cudaMemcpyAsync(g_can, gauge_host, canon_gauge, cudaMemcpyHostToDevice, st))) break;
            if ((s = lqcd_pack_gauge(c, g_nat, g_can, stream)) != LQCD_OK) break;
        }
        for (int i = 0; i < n; ++i) {
            const int k = i % HOST_SLOTS;
            // upload: the slot's previous kernels must have consumed in_can
            if (i >= HOST_SLOTS && fail(cudaStreamWaitEvent(up, comp_done[k], 0))) break;
            if (fail(cudaMemcpyAsync(in_can[k], in_host[i], cb_bytes, cudaMemcpyHostToDevice, up))) break;
            if (fail(cudaEventRecord(in_done[k], up))) break;
            // kernels on the caller's stream: the slot's previous download must have drained out_can
            if (fail(cudaStreamWaitEvent(st, in_done[k], 0))) break;
            if (i >= HOST_SLOTS && fail(cudaStreamWaitEvent(st, out_done[k], 0))) break;
            if ((s = lqcd_pack_spinor(c, in_nat[k], in_can[k], 1 - out_parity[i], stream)) != LQCD_OK) break;
            if ((s = lqcd_dslash_eo(c, out_nat[k], g_nat, in_nat[k], out_parity[i], stream)) != LQCD_OK) break;
            if ((s = lqcd_unpack_spinor(c, out_can[k], out_nat[k], out_parity[i], stream)) != LQCD_OK) break;
            if (fail(cudaEventRecord(comp_done[k], st))) break;
            // download
            if (fail(cudaStreamWaitEvent(down, comp_done[k], 0))) break;
            if (fail(cudaMemcpyAsync(out_host[i], out_can[k], cb_bytes, cudaMemcpyDeviceToHost, down))) break;
            if (fail(cudaEventRecord(out_done[k], down))) break;
        }
    } while (false);
    // drain all three streams before returning (also on the error paths): the results live in host memory
    cudaStreamSynchronize(up);
    cudaStreamSynchronize(down);
    const cudaError_t es = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = es;
    if (s != LQCD_OK) return s;
    return e == cudaSuccess ? LQCD_OK : cuda_fail(e);
}

lqcd_status lqcd_dslash_eo_host(const lqcd_ctx* c, void* out_host, const void* gauge_host, const void* in_host,
                                int out_parity, void* ws, void* stream) {
    if (!out_host || !in_host) return LQCD_EINVAL;
    void* outs[1] = {out_host};
    const void* ins[1] = {in_host};
    return lqcd_dslash_eo_host_batch(c, 1, outs, gauge_host, ins, &out_parity, ws, stream);
}

// ---- next row f4, last clause: pure-gauge heatbath on the update layout of the links (heatbath_kernels.cuh) -----------
size_t lqcd_update_links_bytes(const lqcd_ctx* c) { return c ? (size_t)4 * 2 * 9 * TILE * c->g.ntiles * sizeof(double2) : 0; }

static lqcd_status update_links_convert(const lqcd_ctx* c, void* native, void* canon, void* stream, bool unpack) {
    if (!c || !native || !canon) return LQCD_EINVAL;
    if (c->p.precision != 64) return LQCD_EUNSUPPORTED;   // complex128 links
    if (!aligned16(native) || !aligned16(canon)) return LQCD_EALIGN;
    const dim3 grid((c->g.Vh + HB_BLOCK - 1) / HB_BLOCK, 4, 2);
    if (unpack) update_links_pack_kernel<true><<<grid, HB_BLOCK, 0, (cudaStream_t)stream>>>((double2*)native, (double2*)canon, c->g);
    else update_links_pack_kernel<false><<<grid, HB_BLOCK, 0, (cudaStream_t)stream>>>((double2*)native, (double2*)canon, c->g);
    return after_launch();
}

lqcd_status lqcd_pack_update_links(const lqcd_ctx* c, void* native, const void* canon, void* stream) {
    return update_links_convert(c, native, const_cast<void*>(canon), stream, false);
}

lqcd_status lqcd_unpack_update_links(const lqcd_ctx* c, void* canon, const void* native, void* stream) {
    return update_links_convert(c, const_cast<void*>(native), canon, stream, true);
}

lqcd_status lqcd_reunitarise_links(const lqcd_ctx* c, void* links, void* stream) {
    if (!c || !links) return LQCD_EINVAL;
    if (c->p.precision != 64) return LQCD_EUNSUPPORTED;
    if (!aligned16(links)) return LQCD_EALIGN;
    reunitarise_kernel<<<dim3((c->g.Vh + HB_BLOCK - 1) / HB_BLOCK, 4, 2), HB_BLOCK, 0, (cudaStream_t)stream>>>((double2*)links, c->g);
    return after_launch();
}

size_t lqcd_heatbath_uniforms(const lqcd_ctx* c, int ntries) {
    return c && ntries > 0 ? (size_t)c->g.Vh * 3 * (4 * (size_t)ntries + 2) : 0;
}

lqcd_status lqcd_heatbath_sublattice(const lqcd_ctx* c, void* links, double beta, int mu, int parity, const void* uniforms,
                                     int ntries, void* stream) {
    if (!c || !links || !uniforms) return LQCD_EINVAL;
    if (mu < 0 || mu > 3 || (parity != 0 && parity != 1) || ntries < 1 || ntries > 64 || !(beta > 0.0)) return LQCD_EINVAL;
    if (c->p.precision != 64) return LQCD_EUNSUPPORTED;
    if (!aligned16(links) || (reinterpret_cast<uintptr_t>(uniforms) & 7u)) return LQCD_EALIGN;
    heatbath_kernel<<<(c->g.Vh + HB_BLOCK - 1) / HB_BLOCK, HB_BLOCK, 0, (cudaStream_t)stream>>>(
        (double2*)links, c->g, beta, mu, parity, (const double*)uniforms, ntries);
    return after_launch();
}

size_t lqcd_plaquette_workspace_bytes(const lqcd_ctx* c) {
    return c ? align256((size_t)2 * ((c->g.Vh + HB_BLOCK - 1) / HB_BLOCK) * sizeof(double)) + 256 : 0;
}

lqcd_status lqcd_plaquette(const lqcd_ctx* c, const void* links, void* workspace, double* plaq_host, void* stream) {
    if (!c || !links || !workspace || !plaq_host) return LQCD_EINVAL;
    if (c->p.precision != 64) return LQCD_EUNSUPPORTED;
    if (!aligned16(links) || (reinterpret_cast<uintptr_t>(workspace) & 255u)) return LQCD_EALIGN;
    cudaStream_t st = (cudaStream_t)stream;
    const int nblk = (c->g.Vh + HB_BLOCK - 1) / HB_BLOCK;
    double* partial = static_cast<double*>(workspace);
    double* total = reinterpret_cast<double*>(static_cast<char*>(workspace) + align256((size_t)2 * nblk * sizeof(double)));
    plaquette_kernel<<<dim3(nblk, 2), HB_BLOCK, 0, st>>>((const double2*)links, c->g, partial);
    lqcd_status s = after_launch();
    if (s != LQCD_OK) return s;
    sum_partials_kernel<<<1, BLAS_BLOCK, 0, st>>>(partial, 2 * nblk, total);
    if ((s = after_launch()) != LQCD_OK) return s;
    double sum = 0.0;
    cudaError_t e;
    if ((e = cudaMemcpyAsync(&sum, total, sizeof(double), cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e);
    *plaq_host = sum / (3.0 * 6.0 * 2.0 * (double)c->g.Vh);
    return LQCD_OK;
}

// ---- lqcd_apply_M_eo_static: the even-odd fermion matrix for callers that have no way to allocate device memory ------
// Everything else in this file takes its scratch from the caller.  This one entry point keeps the intermediate odd half
// spinor of M_eo = 1 - kappa^2 H_eo H_oe in an array that is part of the library image itself, so the caller brings only
// out, gauge and in.  The array costs LQCD_STATIC_SCRATCH_BYTES of HBM on every GPU that loads this module, from the
// moment it is loaded until the process exits, whether or not the entry point is ever called -- hence the modest size.
}  // extern "C"

namespace {

constexpr size_t STATIC_SCRATCH_BYTES = LQCD_STATIC_SCRATCH_BYTES;
static __device__ __align__(256) unsigned char g_static_scratch[STATIC_SCRATCH_BYTES];

// In host code `g_static_scratch` is only a handle for the runtime, not an address a kernel may use: the device
// address differs from GPU to GPU and has to be asked for, once per device, with that device current.
constexpr int STATIC_SCRATCH_MAX_DEVICES = 64;
std::mutex g_static_scratch_lock;
void* g_static_scratch_dev[STATIC_SCRATCH_MAX_DEVICES] = {};

lqcd_status static_scratch_address(void** ptr) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e);
    if (dev < 0 || dev >= STATIC_SCRATCH_MAX_DEVICES) return LQCD_EUNSUPPORTED;
    std::lock_guard<std::mutex> guard(g_static_scratch_lock);
    if (!g_static_scratch_dev[dev]) {
        void* p = nullptr;
        if ((e = cudaGetSymbolAddress(&p, g_static_scratch)) != cudaSuccess) return cuda_fail(e);
        g_static_scratch_dev[dev] = p;
    }
    *ptr = g_static_scratch_dev[dev];
    return LQCD_OK;
}

}  // namespace

extern "C" {

size_t lqcd_static_scratch_bytes(void) { return STATIC_SCRATCH_BYTES; }

lqcd_status lqcd_apply_M_eo_static(const lqcd_ctx* c, void* out, const void* gauge, const void* in, double kappa,
                                   void* stream) {
    const size_t hb = c ? half_bytes(c) : 0;
    lqcd_status s = check_fields(c, out, gauge, in, hb);
    if (s != LQCD_OK) return s;
    if (hb > STATIC_SCRATCH_BYTES) return LQCD_ETOOBIG;   // before any CUDA call: the answer does not depend on the device
    void* scratch = nullptr;
    if ((s = static_scratch_address(&scratch)) != LQCD_OK) return s;
    // Nothing in the array has to start from zero: the first launch writes every site of the intermediate field before the
    // second reads it, and the padding lanes of the last tile are neither read nor written.  What an earlier call left
    // behind is simply overwritten.
    return apply_M_impl(c, out, gauge, in, kappa, 0.0, false, 1, scratch, (cudaStream_t)stream);
}

unsigned lqcd_selftest_fastdiv(unsigned d, unsigned n) {
    unsigned mul;
    int shift;
    set_fastdiv(d, mul, shift);
    return fastdiv(n, mul, shift);
}

unsigned long long lqcd_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

const char* lqcd_status_string(lqcd_status s) {
    switch (s) {
        case LQCD_OK: return "ok";
        case LQCD_EINVAL: return "invalid argument";
        case LQCD_EALIGN: return "device pointer not aligned (native fields: 32 bytes, canonical buffers: 16, solver / host workspaces: 256)";
        case LQCD_EALIAS: return "output overlaps an input";
        case LQCD_EUNSUPPORTED: return "unsupported configuration";
        case LQCD_ECUDA: return "CUDA error";
        case LQCD_ETOOBIG: return "lattice too large for the library's built-in scratch array (lqcd_static_scratch_bytes): use the entry point that takes a workspace";
    }
    return "unknown status";
}

const char* lqcd_last_cuda_error(void) { return g_cuda_err; }

}  // extern "C"
