// lstage_kernel.cuh -- the gather kernel with the LINK stream staged through shared memory by the TMA unit.
//
// Same thread -> site map, same arithmetic and the same order as dslash_kernel (bit-identical results); the neighbour
// spinors are gathered into registers as before (their reuse lives in L1).  The links -- two thirds of the bytes, read
// exactly once, contiguous per warp tile and hop in the native layout (fields.cuh: [tile][hop][word][32]) -- no longer
// travel through registers: every warp owns two shared-memory buffers of one UNIT (two hops in fp32, one in fp64:
// 3 KB) and one mbarrier each; its elected lane fetches unit u + 2 with cp.async.bulk as soon as the warp has read unit
// u out of its buffer.  So the link bytes of the next unit are always in flight while the current one is computed on,
// independent of the register budget, and the registers the link words used to occupy while in flight are free for
// deeper spinor gathers.  No producer warps and no cross-warp synchronisation: a warp is the only producer and the
// only consumer of its buffers.  96 KB of shared memory per SM (16 warps x 6 KB), which the gather kernel's L1 use
// tolerates (carve-out sweep: up to 40 % of the 228 KB cost nothing).
#pragma once
#include "pipe_kernel.cuh"

namespace lqcd {

template <typename R, int RECON> struct LStage {
    using P = Pipe<R, RECON>;
    static constexpr int NH = sizeof(R) == 4 ? 2 : 1;          // hops per unit
    static constexpr int UNIT_BYTES = NH * P::LINK_BYTES;
    static constexpr int NU = 8 / NH;                          // units per tile
    static constexpr int WARP_BYTES = 2 * UNIT_BYTES;          // two buffers
    __host__ __device__ static constexpr int smem_bytes(int block) { return (block / 32) * (WARP_BYTES + 16); }
};

// gather + project the neighbour of hop K
template <typename R, int K>
__device__ __forceinline__ void gather_project(const R* __restrict__ in, int nbk, R h[12]) {
    R v[24];
    load_spinor<R>(in, nbk, v);
    project<R, K / 2, (K & 1) ? -1 : +1>(v, h);
}

template <typename R, int RECON, bool CBC, int K>
__device__ __forceinline__ void hop_from_raw(R acc[24], R h[12], const R raw[RECON], unsigned crossmask, const BcPhases<R>& bc) {
    R u[18];
    decode_link<R, RECON>(raw, u);
    hop_rest<R, CBC, K / 2, (K & 1) == 0>(acc, h, (R)1, u, (crossmask >> K) & 1u, bc);
}

// Unit U of the tile: its hops' spinors gathered, its links read from the warp's buffer U & 1, the buffer refilled with
// unit U + 2, then the arithmetic.
template <typename R, int RECON, bool CBC, int U>
__device__ __forceinline__ void lstage_unit(R acc[24], const char* buf, unsigned buf_addr, unsigned bar, const char* tile_links,
                                            const R* __restrict__ in, const int nb[8], unsigned crossmask, const BcPhases<R>& bc,
                                            int lane, unsigned long long evict_first) {
    using L = LStage<R, RECON>;
    constexpr int NH = L::NH, K0 = U * NH;
    R h0[12], h1[12], r0[RECON], r1[RECON];
    gather_project<R, K0>(in, nb[K0], h0);
    if constexpr (NH == 2) gather_project<R, K0 + 1>(in, nb[K0 + 1], h1);
    mbar_wait(bar, (U >> 1) & 1u);
    lds_link<R, RECON>(buf, 0, lane, r0);
    if constexpr (NH == 2) lds_link<R, RECON>(buf, 1, lane, r1);
    if constexpr (U + 2 < L::NU) {
        // The refill may only be issued once every lane's reads of the buffer have returned.  ptxas does not order
        // ld.shared against a later cp.async.bulk into the same bytes (and sinks loads towards their first use, far
        // behind the copy's issue: seen as sporadic wrong sites), and __syncwarp of a converged warp orders nothing;
        // a CTA-scope fence executed by every lane does (MEMBAR waits for the lane's outstanding loads).
        asm volatile("fence.acq_rel.cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) {
            mbar_arrive_expect_tx(bar, L::UNIT_BYTES);
            bulk_copy_hint(buf_addr, tile_links + (U + 2) * L::UNIT_BYTES, L::UNIT_BYTES, bar, evict_first);
        }
    }
    hop_from_raw<R, RECON, CBC, K0>(acc, h0, r0, crossmask, bc);
    if constexpr (NH == 2) hop_from_raw<R, RECON, CBC, K0 + 1>(acc, h1, r1, crossmask, bc);
}

// Launch contract: cb_begin is a multiple of 32 (a warp's sites are one layout tile), R is float or double with links
// of the same precision, dynamic shared memory LStage::smem_bytes(BLOCK).  grid as dslash_kernel.
template <typename R, int RECON, int EPI, bool CBC, int BLOCK>
__global__ void __launch_bounds__(BLOCK, MinBlocks<R, RECON>::value * 64 / BLOCK)
dslash_lstage_kernel(R* __restrict__ out, const R* __restrict__ gauge, const R* __restrict__ in, const R* __restrict__ xin,
                     Epilogue<R> epi, Geom g, int parity0, BcPhases<R> bc, int cb_begin, int cb_end) {
    using L = LStage<R, RECON>;
    using P = Pipe<R, RECON>;
    constexpr bool XPAY = EPI == EPI_XPAY || EPI == EPI_G5XPAY;
    extern __shared__ __align__(128) char smem[];
    int p = parity0;
    if (gridDim.y == 2) {
        p = blockIdx.y;
        const size_t half = half_stride<R>(g.ntiles);
        in += (size_t)(1 - p) * half;
        out += (size_t)p * half;
        if (XPAY) xin += (size_t)p * half;
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int cb_raw = cb_begin + blockIdx.x * BLOCK + threadIdx.x;
    if (cb_raw - lane >= cb_end) return;            // the whole warp is past the range
    const bool live = cb_raw < cb_end;
    const int cb = live ? cb_raw : cb_end - 1;      // dead lanes of a ragged last tile work on a valid site and store nothing
    const int tau = cb_raw >> 5;

    char* const buf = smem + warp * L::WARP_BYTES;
    const unsigned buf_addr = smem_addr(buf);
    const unsigned bar = smem_addr(smem + (BLOCK / 32) * L::WARP_BYTES + warp * 16);
    const char* tile_links = reinterpret_cast<const char*>(gauge) + link_word0<R, RECON>(g.ntiles, p, tau * TILE, 0) * sizeof(typename P::LWd);
    const unsigned long long evict_first = policy_evict_first();
    if (lane == 0) {
        mbar_init(bar, 1);
        mbar_init(bar + 8, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        mbar_arrive_expect_tx(bar, L::UNIT_BYTES);
        bulk_copy_hint(buf_addr, tile_links, L::UNIT_BYTES, bar, evict_first);
        mbar_arrive_expect_tx(bar + 8, L::UNIT_BYTES);
        bulk_copy_hint(buf_addr + L::UNIT_BYTES, tile_links + L::UNIT_BYTES, L::UNIT_BYTES, bar + 8, evict_first);
    }
    __syncwarp();

    const Site s = decode_site(g, cb, p);
    int nb[8];
    unsigned crossmask;
    all_neighbours(g, cb, s, nb, crossmask);
    R acc[24];
#pragma unroll
    for (int k = 0; k < 24; ++k) acc[k] = 0;

#define LQCD_LSTAGE_UNIT(U)                                                                                               \
    if constexpr (U < L::NU)                                                                                              \
        lstage_unit<R, RECON, CBC, U>(acc, buf + (U & 1) * L::UNIT_BYTES, buf_addr + (U & 1) * L::UNIT_BYTES, bar + 8 * (U & 1), \
                                      tile_links, in, nb, crossmask, bc, lane, evict_first);
    LQCD_LSTAGE_UNIT(0) LQCD_LSTAGE_UNIT(1) LQCD_LSTAGE_UNIT(2) LQCD_LSTAGE_UNIT(3)
    LQCD_LSTAGE_UNIT(4) LQCD_LSTAGE_UNIT(5) LQCD_LSTAGE_UNIT(6) LQCD_LSTAGE_UNIT(7)
#undef LQCD_LSTAGE_UNIT

    finish_site<R, EPI>(acc, out, xin, epi, g.ntiles, cb, live);
}

}  // namespace lqcd
