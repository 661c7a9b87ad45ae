// pipe_kernel.cuh -- the Wilson hopping kernel as a persistent, warp-specialised TMA pipeline (north_star (3):
// "shared-memory or TMA staging of neighbour tiles chosen for Blackwell's L2 and SMEM").
//
// Same arithmetic as dslash_kernel (steps K1-K6 of SURVEY.md sec. 8(a); "the non-diagonal part of the
// Dirac matrix ('dslash')"), in the same order, so the results are bit-identical; different data movement.
// dslash_kernel keeps every operand in flight in registers: a thread alternates between waiting for its gathers and
// computing on them.  Here the two are decoupled:
//
//   * one CTA per SM, resident for the whole launch; work unit = one warp tile (32 consecutive checkerboard sites);
//     CTA b processes the tiles b, b + gridDim.x, ... of the launch's range;
//   * warps 0..3 (the producers, one per direction mu) stage every tile's operands in four rings of shared-memory
//     slots with cp.async.bulk (the TMA unit's linear copies; completion is counted on an mbarrier per slot); lanes
//     0..3 each compute the address of one copy and issue it.  Chunk mu of a tile holds the links of hops 2 mu and
//     2 mu + 1 of its 32 sites -- contiguous in the native layout (fields.cuh: [tile][hop][word][32]) -- and whole
//     tiles of the input field:
//        X  the tile itself (the x neighbours of site cb are cb and cb +- 1);
//        Y  the tile holding the -y neighbour of the first lane, the tile itself, the tile holding the +y neighbour
//           of the last lane;
//        Z, T  the two tiles holding the forward / backward neighbour of the first lane.
//     On lattices whose z planes are multiples of 32 sites (all bench sizes) a z or t neighbour tile is exactly the
//     neighbours of the 32 lanes, in lane order;
//   * the other warps (the consumers) each take every NC-th tile of the CTA: for each direction wait until the chunk
//     has landed, read the two neighbour spinors (projecting them at once) and the two links with LDS, release the
//     slot, and do the arithmetic of the two hops from registers; after the T chunk the epilogue and the store
//     (finish_site).  A lane whose neighbour is in none of the staged tiles (rows that wrap around the lattice
//     inside a tile, lattices with small or odd-sized planes) gathers it from global memory exactly as dslash_kernel
//     does -- every geometry is handled, the regular ones without a single gather.
//
// Each ring is a FIFO in tile order.  A slot carries an mbarrier ("full": the chunk's bytes have landed) and a counter
// of the uses released so far (a consumer's store-release once its reads are in registers).  Different warps
// consume the successive uses of one slot, and an mbarrier wait only knows the parity of a phase, so nobody touches a
// slot for use u before the counter says that use u - 1 is over: the producer to refill it, the consumer before it
// waits on "full".  A slot is held for the landing time of its chunk plus a few dozen LDS, so a handful of slots per
// ring keeps the memory system busy whatever the consumers are doing: bytes in flight per SM are bounded by the rings
// (~200 KB), not by registers and resident warps.
#pragma once
#include "dslash_kernel.cuh"

namespace lqcd {

// ---- mbarrier / bulk-copy primitives --------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// try_wait suspends the thread in hardware until the phase completes or the time hint (ns) runs out
#ifndef LQCD_PIPE_WAIT_HINT_NS
#define LQCD_PIPE_WAIT_HINT_NS 1000
#endif
__device__ __forceinline__ bool mbar_try_wait(unsigned bar, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2, %3;\n"
        "selp.u32 %0, 1, 0, P1;\n"
        "}" : "=r"(ok) : "r"(bar), "r"(parity), "r"((unsigned)LQCD_PIPE_WAIT_HINT_NS) : "memory");
    return ok != 0;
}
// Bounded: a pipeline bug traps the kernel after a few seconds instead of hanging the GPU.  The clock is only looked
// at every 4096 failed attempts (the inner loop is nothing but the try_wait).
static __device__ __noinline__ void mbar_wait_slow(unsigned bar, unsigned parity) {
    unsigned long long t0, t1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    for (;;) {
        for (int n = 0; n < 4096; ++n)
            if (mbar_try_wait(bar, parity)) return;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
        if (t1 - t0 > 4000000000ull) __trap();
    }
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    if (mbar_try_wait(bar, parity)) return;
    if (mbar_try_wait(bar, parity)) return;
    mbar_wait_slow(bar, parity);
}
// global -> shared linear copy by the TMA unit; `bytes` (a multiple of 16) are counted on `bar` when they have landed
__device__ __forceinline__ void bulk_copy(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_copy_hint(unsigned dst, const void* src, unsigned bytes, unsigned bar, unsigned long long policy) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(policy) : "memory");
}
// one lane of the (converged) warp; the region it guards is single-threaded, so copies issue straight from uniform registers
__device__ __forceinline__ bool elect_one() {
    unsigned pred;
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "elect.sync _|P1, 0xffffffff;\n"
        "selp.u32 %0, 1, 0, P1;\n"
        "}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ unsigned long long policy_evict_first() {
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}

// ---- sizes ------------------------------------------------------------------------------------------------------------
// consumer warps per CTA (plus 4 producer warps).  fp32: 4 + 12 warps of 128 registers; fp64: 4 + 8 warps of 168.
#ifndef LQCD_PIPE_CONSUMERS_F32
#define LQCD_PIPE_CONSUMERS_F32 12
#endif
#ifndef LQCD_PIPE_CONSUMERS_F64
#define LQCD_PIPE_CONSUMERS_F64 8
#endif
template <typename R, int RECON> struct Pipe {
    using LWd = typename LinkWord<R, RECON>::type;
    static constexpr int LW = LinkWord<R, RECON>::LW, NW = RECON / LW;
    static constexpr int W = Word<R>::W, Q = 24 / W;
    static constexpr int LINK_BYTES = NW * TILE * (int)sizeof(LWd);   // the links of one hop of a tile
    static constexpr int TILE_BYTES = Q * TILE * 32;                  // one tile of a half spinor
    // chunk of direction mu: links of hops 2 mu, 2 mu + 1 | NTILES(mu) staged tiles
    __host__ __device__ static constexpr int ntiles(int mu) { return mu == 0 ? 1 : (mu == 1 ? 3 : 2); }
    __host__ __device__ static constexpr int chunk_bytes(int mu) { return 2 * LINK_BYTES + ntiles(mu) * TILE_BYTES; }
    static constexpr int TILE_SET_BYTES = chunk_bytes(0) + chunk_bytes(1) + chunk_bytes(2) + chunk_bytes(3);
    static constexpr int BAR_BYTES = 1024;                            // full[mu][slot] (mbarriers), released[mu][slot] (u32)
    static constexpr int SMEM_MAX = 227 * 1024;
    static constexpr int DEPTH = (SMEM_MAX - BAR_BYTES) / TILE_SET_BYTES;   // slots per ring
    __host__ __device__ static constexpr int ring_offset(int mu) {
        return BAR_BYTES + DEPTH * (mu == 0 ? 0 : (mu == 1 ? chunk_bytes(0) : (mu == 2 ? chunk_bytes(0) + chunk_bytes(1)
                                                                                       : chunk_bytes(0) + chunk_bytes(1) + chunk_bytes(2))));
    }
    static constexpr int SMEM_BYTES = BAR_BYTES + DEPTH * TILE_SET_BYTES;
    static constexpr int NP = 4;
    static constexpr int NC = sizeof(R) == 4 ? LQCD_PIPE_CONSUMERS_F32 : LQCD_PIPE_CONSUMERS_F64;
    static constexpr int THREADS = 32 * (NP + NC);
    static_assert(LINK_BYTES % 128 == 0 && 4 * DEPTH * 12 <= BAR_BYTES && DEPTH >= 2, "slot layout");
};

// a spinor from a staged tile in shared memory: word q of position pos at buf + q * 1024 + pos * 32
template <typename R>
__device__ __forceinline__ void lds_spinor(const char* buf, int pos, R v[24]) {
    constexpr int W = Word<R>::W, Q = 24 / W;
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        const char* p = buf + q * (TILE * 32) + pos * 32;
        if constexpr (sizeof(R) == 4) {
            const float4 a = *reinterpret_cast<const float4*>(p), b = *reinterpret_cast<const float4*>(p + 16);
            v[q * W + 0] = a.x; v[q * W + 1] = a.y; v[q * W + 2] = a.z; v[q * W + 3] = a.w;
            v[q * W + 4] = b.x; v[q * W + 5] = b.y; v[q * W + 6] = b.z; v[q * W + 7] = b.w;
        } else {
            const double2 a = *reinterpret_cast<const double2*>(p), b = *reinterpret_cast<const double2*>(p + 16);
            v[q * W + 0] = a.x; v[q * W + 1] = a.y; v[q * W + 2] = b.x; v[q * W + 3] = b.y;
        }
    }
}

// the stored reals of the kk-th link block of a chunk, for this lane's site
template <typename R, int RECON>
__device__ __forceinline__ void lds_link(const char* links, int kk, int lane, R raw[RECON]) {
    using P = Pipe<R, RECON>;
    using LWd = typename P::LWd;
    const LWd* p = reinterpret_cast<const LWd*>(links + kk * P::LINK_BYTES) + lane;
#pragma unroll
    for (int w = 0; w < P::NW; ++w) {
        const LWd x = p[w * TILE];
        unpack(x, raw + w * P::LW);
    }
}

// K2 on the stored reals
template <typename R, int RECON>
__device__ __forceinline__ void decode_link(const R raw[RECON], R u[18]) {
    if constexpr (RECON == 8) {
        recon8<R>(raw, u);
    } else {
#pragma unroll
        for (int k = 0; k < RECON; ++k) u[k] = raw[k];
        if constexpr (RECON == 12) recon_row2<R>(u);
    }
}

// The slot's use counter (see the header): wait until `use` uses have been released.  Bounded like mbar_wait.
__device__ __forceinline__ bool released_reached(unsigned released, unsigned use) {
    unsigned v;
    asm volatile("ld.acquire.cta.shared.u32 %0, [%1];" : "=r"(v) : "r"(released) : "memory");
    return v >= use;
}
static __device__ __noinline__ void await_released_slow(unsigned released, unsigned use) {
    unsigned long long t0, t1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    for (;;) {
        for (int n = 0; n < 4096; ++n) {
            if (released_reached(released, use)) return;
            __nanosleep(20);
        }
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
        if (t1 - t0 > 4000000000ull) __trap();
    }
}
__device__ __forceinline__ void await_released(unsigned released, unsigned use) {
    if (use == 0 || released_reached(released, use)) return;
    await_released_slow(released, use);
}

// Consumer side.  The four directions of a tile are ONE loop body executed four times (not four unrolled copies): the
// consumer warps of an SM sit at different places of the tile loop, so the code they run must stay small enough for
// the instruction caches (an unrolled body is 28 KB of straight-line code per precision and starved 12 desynchronised
// warps of instructions: ncu stall_no_inst).  Only what really depends on the direction -- where the neighbours are
// staged, the projection K3 and the reconstruction K5 -- is dispatched on mu; the loads, the link reconstruction K2 and
// the colour multiply K4 are shared code.
struct StagedOperand { const char* buf; int pos; int nb; };   // pos >= 0: position in the staged tile `buf`; else gather site nb

template <typename R, int RECON, int MU>
__device__ __forceinline__ void locate_operands(StagedOperand& f, StagedOperand& b, const char* slot, int tau, const int nb[8]) {
    using P = Pipe<R, RECON>;
    const int nf = nb[2 * MU], nk = nb[2 * MU + 1];
    const char* tiles = slot + 2 * P::LINK_BYTES;
    f.nb = nf;
    b.nb = nk;
    if constexpr (MU == 0) {          // the tile itself
        f.buf = b.buf = tiles;
        f.pos = (nf >> 5) == tau ? (nf & 31) : -1;
        b.pos = (nk >> 5) == tau ? (nk & 31) : -1;
    } else if constexpr (MU == 1) {   // [tile of lane 0's -y neighbour | the tile itself | tile of lane 31's +y neighbour]
        const int ta = __shfl_sync(0xffffffffu, nk, 0) >> 5, tc = __shfl_sync(0xffffffffu, nf, 31) >> 5;
        const int tf = nf >> 5, tb = nk >> 5;
        f.pos = (tf == tau || tf == ta || tf == tc) ? (nf & 31) : -1;
        b.pos = (tb == tau || tb == ta || tb == tc) ? (nk & 31) : -1;
        f.buf = tiles + (tf == tau ? 1 : (tf == ta ? 0 : 2)) * P::TILE_BYTES;
        b.buf = tiles + (tb == tau ? 1 : (tb == ta ? 0 : 2)) * P::TILE_BYTES;
    } else {                          // [tile of lane 0's forward neighbour | tile of its backward neighbour]
        const int tf = __shfl_sync(0xffffffffu, nf, 0) >> 5, tb = __shfl_sync(0xffffffffu, nk, 0) >> 5;
        f.buf = tiles;
        b.buf = tiles + P::TILE_BYTES;
        f.pos = (nf >> 5) == tf ? (nf & 31) : -1;
        b.pos = (nk >> 5) == tb ? (nk & 31) : -1;
    }
}

template <typename R>
__device__ __forceinline__ void fetch_spinor(const StagedOperand& o, const R* __restrict__ in, R v[24]) {
    if (o.pos >= 0) lds_spinor<R>(o.buf, o.pos, v); else load_spinor<R>(in, o.nb, v);
}

template <typename R, int S>
__device__ __forceinline__ void project_mu(int mu, const R v[24], R h[12]) {
    switch (mu) {
        case 0: project<R, 0, S>(v, h); break;
        case 1: project<R, 1, S>(v, h); break;
        case 2: project<R, 2, S>(v, h); break;
        default: project<R, 3, S>(v, h); break;
    }
}
template <typename R, int S>
__device__ __forceinline__ void reconstruct_accumulate_mu(int mu, R acc[24], const R chi[12], R f) {
    switch (mu) {
        case 0: reconstruct_accumulate<R, 0, S>(acc, chi, f); break;
        case 1: reconstruct_accumulate<R, 1, S>(acc, chi, f); break;
        case 2: reconstruct_accumulate<R, 2, S>(acc, chi, f); break;
        default: reconstruct_accumulate<R, 3, S>(acc, chi, f); break;
    }
}

// acc = (H in)(x) for this lane's site of tile tau: the chunks of the four directions out of ring slot sl, use `use`
template <typename R, int RECON, bool CBC>
__device__ __forceinline__ void consume_tile(R acc[24], char* smem, unsigned bars, unsigned rels, unsigned sl, unsigned use,
                                             const R* __restrict__ in, int lane, int tau, const int nb[8], unsigned crossmask,
                                             const BcPhases<R>& bc) {
    using P = Pipe<R, RECON>;
#pragma unroll 1
    for (int mu = 0; mu < 4; ++mu) {
        StagedOperand of, ob;
        const char* slot;
        R br, bi;
        switch (mu) {
            case 0: slot = smem + P::ring_offset(0) + sl * P::chunk_bytes(0); locate_operands<R, RECON, 0>(of, ob, slot, tau, nb); br = bc.re[0]; bi = bc.im[0]; break;
            case 1: slot = smem + P::ring_offset(1) + sl * P::chunk_bytes(1); locate_operands<R, RECON, 1>(of, ob, slot, tau, nb); br = bc.re[1]; bi = bc.im[1]; break;
            case 2: slot = smem + P::ring_offset(2) + sl * P::chunk_bytes(2); locate_operands<R, RECON, 2>(of, ob, slot, tau, nb); br = bc.re[2]; bi = bc.im[2]; break;
            default: slot = smem + P::ring_offset(3) + sl * P::chunk_bytes(3); locate_operands<R, RECON, 3>(of, ob, slot, tau, nb); br = bc.re[3]; bi = bc.im[3]; break;
        }
        const unsigned full_bar = bars + 8 * (mu * P::DEPTH + sl), released = rels + 4 * (mu * P::DEPTH + sl);
        // my turn on this slot (its previous use is over), then the data
        if (lane == 0) await_released(released, use);
        __syncwarp();
        mbar_wait(full_bar, use & 1u);
        R hf[12], hb[12], rf[RECON], rb[RECON];
        {
            R v[24];
            fetch_spinor<R>(of, in, v);
            project_mu<R, +1>(mu, v, hf);
            fetch_spinor<R>(ob, in, v);
            project_mu<R, -1>(mu, v, hb);
        }
        lds_link<R, RECON>(slot, 0, lane, rf);
        lds_link<R, RECON>(slot, 1, lane, rb);
        __syncwarp();                             // every lane's shared-memory reads of the chunk are in registers
        if (lane == 0) asm volatile("st.release.cta.shared.u32 [%0], %1;" ::"r"(released), "r"(use + 1u) : "memory");
        R u[18], chi[12];
        const unsigned cross = crossmask >> (2 * mu);
        decode_link<R, RECON>(rf, u);
        R f = boundary_phase<R, CBC>(hf, (R)1, cross & 1u, br, bi);
        su3_multiply<R, true>(hf, u, chi);
        reconstruct_accumulate_mu<R, +1>(mu, acc, chi, f);
        decode_link<R, RECON>(rb, u);
        f = boundary_phase<R, CBC>(hb, (R)1, (cross >> 1) & 1u, br, -bi);
        su3_multiply<R, false>(hb, u, chi);
        reconstruct_accumulate_mu<R, -1>(mu, acc, chi, f);
    }
}

// Producer warp of direction MU.  Every lane computes the same (warp-uniform) addresses; one elected lane waits for the
// slot, arms the barrier and issues the copies: the link block of hops 2 MU, 2 MU + 1, then the staged tiles.
template <typename R, int RECON, int MU>
__device__ __forceinline__ void produce_direction(char* smem, unsigned bars, unsigned rels, const R* __restrict__ gauge, const R* __restrict__ in,
                                                  const Geom& g, int parity0, int both, int tile0, int nt, int n_mine, size_t half) {
    using P = Pipe<R, RECON>;
    const unsigned long long evict_first = policy_evict_first();
    const unsigned ring = smem_addr(smem) + (unsigned)P::ring_offset(MU);
    unsigned slot = 0, use = 0;
    for (int i = 0; i < n_mine; ++i) {
        const int j = blockIdx.x + i * gridDim.x;
        const int pj = both ? j / nt : 0, tau = tile0 + (j - pj * nt);
        const int p = both ? pj : parity0;
        const char* in_p = reinterpret_cast<const char*>(both ? in + (size_t)(1 - p) * half : in);
        const char* links = reinterpret_cast<const char*>(gauge) + link_word0<R, RECON>(g.ntiles, p, tau * TILE, 2 * MU) * sizeof(typename P::LWd);
        // staged tiles t0, t1, t2 -> buffers 0, 1, 2 (-1: nothing to copy)
        int t0 = tau, t1 = -1, t2 = -1;
        if constexpr (MU != 0) {
            bool c;
            const int first = min(tau * TILE, g.Vh - 1);
            const Site sf = decode_site(g, first, p);
            if constexpr (MU == 1) {
                const int lastc = min(tau * TILE + TILE - 1, g.Vh - 1);
                const Site sl = decode_site(g, lastc, p);
                const int a = neighbour<1, false>(g, first, sf, c) >> 5, cc = neighbour<1, true>(g, lastc, sl, c) >> 5;
                t0 = a != tau ? a : -1;                 // tile of the first lane's -y neighbour
                t1 = tau;                               // the tile itself
                t2 = (cc != tau && cc != a) ? cc : -1;  // tile of the last lane's +y neighbour
            } else {
                t0 = neighbour<MU, true>(g, first, sf, c) >> 5;
                t1 = neighbour<MU, false>(g, first, sf, c) >> 5;
            }
        }
        const unsigned dst = ring + slot * (unsigned)P::chunk_bytes(MU), tiles = dst + 2 * P::LINK_BYTES;
        const unsigned full = bars + 8 * (MU * P::DEPTH + slot), released = rels + 4 * (MU * P::DEPTH + slot);
        if (elect_one()) {
            await_released(released, use);        // the slot's previous chunk has been consumed
            mbar_arrive_expect_tx(full, 2 * P::LINK_BYTES + ((t0 >= 0) + (t1 >= 0) + (t2 >= 0)) * P::TILE_BYTES);
            bulk_copy_hint(dst, links, 2 * P::LINK_BYTES, full, evict_first);   // links are read once per application
            if (t0 >= 0) bulk_copy(tiles, in_p + (size_t)t0 * P::TILE_BYTES, P::TILE_BYTES, full);
            if (t1 >= 0) bulk_copy(tiles + P::TILE_BYTES, in_p + (size_t)t1 * P::TILE_BYTES, P::TILE_BYTES, full);
            if (t2 >= 0) bulk_copy(tiles + 2 * P::TILE_BYTES, in_p + (size_t)t2 * P::TILE_BYTES, P::TILE_BYTES, full);
        }
        __syncwarp();
        if (++slot == P::DEPTH) { slot = 0; ++use; }
    }
}

// out = epilogue(H in) on the sites [cb_begin, cb_end) of parity parity0 (both = 0) or of both parities (both = 1:
// in / out / xin are full fields [even | odd]).  grid.x persistent CTAs of 4 + NC warps.
template <typename R, int RECON, int EPI, bool CBC>
__global__ void __launch_bounds__(Pipe<R, RECON>::THREADS, 1)
dslash_pipe_kernel(R* __restrict__ out, const R* __restrict__ gauge, const R* __restrict__ in, const R* __restrict__ xin,
                   Epilogue<R> epi, Geom g, int parity0, int both, BcPhases<R> bc, int cb_begin, int cb_end) {
    using P = Pipe<R, RECON>;
    extern __shared__ __align__(1024) char smem[];
    // full[mu][s] at 8 (mu DEPTH + s): mbarriers; released[mu][s]: u32 use counters behind them
    const unsigned bars = smem_addr(smem);
    const unsigned rels = bars + 8 * 4 * P::DEPTH;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int s = 0; s < 4 * P::DEPTH; ++s) {
            mbar_init(bars + 8 * s, 1);
            asm volatile("st.shared.u32 [%0], %1;" ::"r"(rels + 4 * s), "r"(0u) : "memory");
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // tiles of the range, per parity; work item j = (parity index, tile) -> this CTA takes j = blockIdx.x + i gridDim.x
    const int tile0 = cb_begin >> 5;
    const int nt = ((cb_end + TILE - 1) >> 5) - tile0;
    const int nwork = both ? 2 * nt : nt;
    const int n_mine = (int)blockIdx.x < nwork ? (nwork - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
    const size_t half = half_stride<R>(g.ntiles);

    if (warp < P::NP) {
        // ---- producers: warp mu stages the chunks of direction mu ----
        switch (warp) {
            case 0: produce_direction<R, RECON, 0>(smem, bars, rels, gauge, in, g, parity0, both, tile0, nt, n_mine, half); break;
            case 1: produce_direction<R, RECON, 1>(smem, bars, rels, gauge, in, g, parity0, both, tile0, nt, n_mine, half); break;
            case 2: produce_direction<R, RECON, 2>(smem, bars, rels, gauge, in, g, parity0, both, tile0, nt, n_mine, half); break;
            default: produce_direction<R, RECON, 3>(smem, bars, rels, gauge, in, g, parity0, both, tile0, nt, n_mine, half); break;
        }
    } else {
        // ---- consumers ----
        const int w = warp - P::NP;
        for (int i = w; i < n_mine; i += P::NC) {
            const int j = blockIdx.x + i * gridDim.x;
            const int pj = both ? j / nt : 0, tau = tile0 + (j - pj * nt);
            const int p = both ? pj : parity0;
            const R* in_p = both ? in + (size_t)(1 - p) * half : in;
            R* out_p = both ? out + (size_t)p * half : out;
            const R* xin_p = (both && xin) ? xin + (size_t)p * half : xin;
            const int cb_raw = tau * TILE + lane;
            const bool live = cb_raw >= cb_begin && cb_raw < cb_end;
            const int cb = min(cb_raw, g.Vh - 1);
            const Site s = decode_site(g, cb, p);
            int nb[8];
            unsigned crossmask;
            all_neighbours(g, cb, s, nb, crossmask);
            R acc[24];
#pragma unroll
            for (int k = 0; k < 24; ++k) acc[k] = 0;
            consume_tile<R, RECON, CBC>(acc, smem, bars, rels, (unsigned)i % P::DEPTH, (unsigned)i / P::DEPTH, in_p, lane, tau, nb, crossmask, bc);
            finish_site<R, EPI>(acc, out_p, xin_p, epi, g.ntiles, cb, live);
        }
    }
}

}  // namespace lqcd
