// slab_kernels.cuh -- time-slab decomposition of the even-odd dslash over several GPUs (next row f3).
//
// The paper's multi-device story is host-mediated ("synchronize the physical gauge field when it is used on several
// devices"; tasks on several devices).  Here a rank owns T_loc consecutive time slices
// (T_loc even, so local and global site parities agree) as a local lattice of exactly those slices.  The only data a
// dslash needs from a neighbouring rank are the two boundary time slices of the input field, and of those only the
// spin-projected half: the forward t hop uses (1 - gamma_t) psi = (psi0 + psi2, psi1 + psi3), the backward one
// (1 + gamma_t) psi = (psi0 - psi2, psi1 - psi3) -- 12 reals per face site instead of 24.
//
//   face_project_kernel   projects the first / last time slice of `in` and stores the half spinors straight into the
//                         destination buffers -- the neighbours' halo buffers, mapped into this GPU's address space over
//                         NVLink (peer memory), or local send buffers when the transport is ncclSend/Recv
//   face_signal_kernel    one thread: system-scope release of the epoch into the neighbours' flags (peer memory)
//   dslash_slab_kernel    dslash_kernel for a range of time slices whose t hops leaving the slab read the halo buffers;
//                         optionally waits (system-scope acquire) on the flags first, so projection, transfer and the
//                         boundary sites need no host round trip; the interior slices are plain lqcd_dslash_eo_range
//
// Halo buffer: [face tile][word][32] 16-byte words (float4 / double2), 3 (fp32) or 6 (fp64) words per site, face site
// f = checkerboard index within the time slice; tiles of 32, the last one padded.
#pragma once
#include "dslash_kernel.cuh"

namespace lqcd {

template <typename R> struct HaloWord;
template <> struct HaloWord<float>  { using type = float4;  static constexpr int W = 4, NW = 3; };
template <> struct HaloWord<double> { using type = double2; static constexpr int W = 2, NW = 6; };

__host__ __device__ __forceinline__ int face_tiles(const Geom& g) { return (g.st + TILE - 1) / TILE; }

template <typename R>
__device__ __forceinline__ void store_half(R* __restrict__ halo, int f, const R h[12]) {
    using Wd = typename HaloWord<R>::type;
    constexpr int W = HaloWord<R>::W, NW = HaloWord<R>::NW;
    Wd* p = reinterpret_cast<Wd*>(halo) + (size_t)(f / TILE) * (NW * TILE) + (f % TILE);
#pragma unroll
    for (int w = 0; w < NW; ++w) {
        Wd x;
        if constexpr (W == 4) x = make_float4(h[4 * w], h[4 * w + 1], h[4 * w + 2], h[4 * w + 3]);
        else x = make_double2(h[2 * w], h[2 * w + 1]);
        p[w * TILE] = x;   // plain st.global: the destination may be peer memory
    }
}

// Halo words are written by another GPU (or another stream) possibly while this kernel is already resident: read them
// through L2 (ld.global.cg), never through the read-only path.
template <typename R>
__device__ __forceinline__ void load_half(const R* halo, int f, R h[12]) {
    using Wd = typename HaloWord<R>::type;
    constexpr int W = HaloWord<R>::W, NW = HaloWord<R>::NW;
    const Wd* p = reinterpret_cast<const Wd*>(halo) + (size_t)(f / TILE) * (NW * TILE) + (f % TILE);
#pragma unroll
    for (int w = 0; w < NW; ++w) {
        const Wd x = __ldcg(p + w * TILE);
        if constexpr (W == 4) { h[4 * w] = x.x; h[4 * w + 1] = x.y; h[4 * w + 2] = x.z; h[4 * w + 3] = x.w; }
        else { h[2 * w] = x.x; h[2 * w + 1] = x.y; }
    }
}

// grid: (ceil(st / block), 2).  blockIdx.y = 0: the LAST time slice, projected with (1 + gamma_t) for the backward hop of
// the rank above (-> dst_up);  blockIdx.y = 1: the FIRST time slice, projected with (1 - gamma_t) for the forward hop of
// the rank below (-> dst_down).  `in` holds the sites of one parity; face site f is cb = t * st + f.
template <typename R>
__global__ void __launch_bounds__(128) face_project_kernel(const R* __restrict__ in, R* __restrict__ dst_up, R* __restrict__ dst_down, Geom g) {
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= g.st) return;
    R v[24], h[12];
    if (blockIdx.y == 0) {
        if (!dst_up) return;
        load_spinor<R>(in, (g.T - 1) * g.st + f, v);
        project<R, 3, -1>(v, h);
        store_half<R>(dst_up, f, h);
    } else {
        if (!dst_down) return;
        load_spinor<R>(in, f, v);
        project<R, 3, +1>(v, h);
        store_half<R>(dst_down, f, h);
    }
}

// After face_project_kernel on the same stream: make its (peer) stores visible system-wide, then publish the epoch.
static __global__ void face_signal_kernel(unsigned long long* flag_up, unsigned long long* flag_down, unsigned long long epoch) {
    __threadfence_system();
    if (flag_up) asm volatile("st.release.sys.global.u64 [%0], %1;" ::"l"(flag_up), "l"(epoch) : "memory");
    if (flag_down) asm volatile("st.release.sys.global.u64 [%0], %1;" ::"l"(flag_down), "l"(epoch) : "memory");
}

// Wait until *flag >= epoch (written by the neighbour's face_signal_kernel).  Bounded: a neighbour that never signals
// (a bug, or a dead rank) traps this kernel after ~10 s instead of hanging the GPU.
__device__ __forceinline__ void wait_flag(const unsigned long long* flag, unsigned long long epoch) {
    unsigned long long t0, t1, v;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    for (;;) {
        asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(flag) : "memory");
        if (v >= epoch) return;
        __nanosleep(200);
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
        if (t1 - t0 > 10000000000ull) __trap();
    }
}

// One of the two t hops of a slab site: from the halo if the hop leaves the slab, gathered otherwise.
template <typename R, int RECON, bool CBC, bool FWD>
__device__ __forceinline__ void hop_t_slab(R acc[24], const typename LinkStore<R, RECON>::word* __restrict__ site_links,
                                           const R* __restrict__ in, const R* halo, bool from_halo, int f, int nb, bool cross,
                                           const BcPhases<R>& bc) {
    R h[12], u[18];
    if (from_halo) {
        load_half<R>(halo, f, h);
    } else {
        R v[24];
        load_spinor<R>(in, nb, v);
        project<R, 3, FWD ? +1 : -1>(v, h);
    }
    load_link<R, RECON>(site_links, FWD ? 6 : 7, u);
    hop_rest<R, CBC, 3, FWD>(acc, h, (R)1, u, cross, bc);
}

// out = H in on the sites [cb_begin, cb_end) of parity p of a slab; one thread per site, EPI_STORE only.
template <typename R, int RECON, bool CBC, int BLOCK>
__global__ void __launch_bounds__(BLOCK, MinBlocks<R, RECON>::value * 64 / BLOCK)
dslash_slab_kernel(R* __restrict__ out, const R* __restrict__ gauge, const R* __restrict__ in, const R* halo_from_up,
                   const R* halo_from_down, const unsigned long long* wait_up, const unsigned long long* wait_down,
                   unsigned long long epoch, Geom g, int p, BcPhases<R> bc, int cb_begin, int cb_end) {
    if (wait_up || wait_down) {
        if (threadIdx.x == 0) {
            if (wait_up) wait_flag(wait_up, epoch);
            if (wait_down) wait_flag(wait_down, epoch);
        }
        __syncthreads();
    }
    const int cb = cb_begin + blockIdx.x * BLOCK + threadIdx.x;
    if (cb >= cb_end) return;
    const Site s = decode_site(g, cb, p);
    int nb[8];
    unsigned crossmask;
    all_neighbours(g, cb, s, nb, crossmask);
    const auto* site_links = reinterpret_cast<const typename LinkStore<R, RECON>::word*>(gauge) +
                             LinkStore<R, RECON>::word0(g.ntiles, p, cb, 0);
    R acc[24];
#pragma unroll
    for (int k = 0; k < 24; ++k) acc[k] = 0;
    hop_step<R, RECON, CBC, 0>(acc, site_links, in, g.ntiles, nb, crossmask, bc);
    hop_step<R, RECON, CBC, 1>(acc, site_links, in, g.ntiles, nb, crossmask, bc);
    hop_step<R, RECON, CBC, 2>(acc, site_links, in, g.ntiles, nb, crossmask, bc);
    hop_step<R, RECON, CBC, 3>(acc, site_links, in, g.ntiles, nb, crossmask, bc);
    hop_step<R, RECON, CBC, 4>(acc, site_links, in, g.ntiles, nb, crossmask, bc);
    hop_step<R, RECON, CBC, 5>(acc, site_links, in, g.ntiles, nb, crossmask, bc);
    const int f = cb - s.t * g.st;   // index within the time slice = face site of the neighbour straight above / below
    hop_t_slab<R, RECON, CBC, true>(acc, site_links, in, halo_from_up, s.t == g.T - 1, f, nb[6], (crossmask >> 6) & 1u, bc);
    hop_t_slab<R, RECON, CBC, false>(acc, site_links, in, halo_from_down, s.t == 0, f, nb[7], (crossmask >> 7) & 1u, bc);
    store_spinor<R>(out, cb, acc);
}

}  // namespace lqcd
