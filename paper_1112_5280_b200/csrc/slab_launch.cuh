// slab_launch.cuh -- host-side launchers of the time-slab kernels (slab_kernels.cuh), instantiated per precision in
// inst_slab_f32.cu / inst_slab_f64.cu and called from lqcd.cu.
#pragma once
#include "launch.cuh"
#include "slab_kernels.cuh"

namespace lqcd {

template <typename R, int RECON>
lqcd_status launch_slab_recon(const lqcd_ctx* c, void* out, const void* gauge, const void* in, const void* halo_up,
                              const void* halo_down, const unsigned long long* wait_up, const unsigned long long* wait_down,
                              unsigned long long epoch, int parity, cudaStream_t st, CbRange rg) {
    constexpr int BLOCK = DSLASH_BLOCK;
    const unsigned grid = (rg.end - rg.begin + BLOCK - 1) / BLOCK;
    if (c->complex_bc)
        dslash_slab_kernel<R, RECON, true, BLOCK><<<grid, BLOCK, 0, st>>>((R*)out, (const R*)gauge, (const R*)in, (const R*)halo_up,
            (const R*)halo_down, wait_up, wait_down, epoch, c->g, parity, make_bc<R>(c), rg.begin, rg.end);
    else
        dslash_slab_kernel<R, RECON, false, BLOCK><<<grid, BLOCK, 0, st>>>((R*)out, (const R*)gauge, (const R*)in, (const R*)halo_up,
            (const R*)halo_down, wait_up, wait_down, epoch, c->g, parity, make_bc<R>(c), rg.begin, rg.end);
    return after_launch();
}

template <typename R>
lqcd_status launch_slab(const lqcd_ctx* c, void* out, const void* gauge, const void* in, const void* halo_up,
                        const void* halo_down, const unsigned long long* wait_up, const unsigned long long* wait_down,
                        unsigned long long epoch, int parity, cudaStream_t st, CbRange rg) {
    switch (c->p.recon) {
        case 8: return launch_slab_recon<R, 8>(c, out, gauge, in, halo_up, halo_down, wait_up, wait_down, epoch, parity, st, rg);
        case 12: return launch_slab_recon<R, 12>(c, out, gauge, in, halo_up, halo_down, wait_up, wait_down, epoch, parity, st, rg);
        case 18: return launch_slab_recon<R, 18>(c, out, gauge, in, halo_up, halo_down, wait_up, wait_down, epoch, parity, st, rg);
    }
    return LQCD_EUNSUPPORTED;
}

template <typename R>
lqcd_status launch_push_faces(const lqcd_ctx* c, const void* in, void* dst_up, void* dst_down, unsigned long long* flag_up,
                              unsigned long long* flag_down, unsigned long long epoch, cudaStream_t st) {
    const dim3 grid((c->g.st + 127) / 128, 2);
    face_project_kernel<R><<<grid, 128, 0, st>>>((const R*)in, (R*)dst_up, (R*)dst_down, c->g);
    lqcd_status s = after_launch();
    if (s != LQCD_OK || (!flag_up && !flag_down)) return s;
    face_signal_kernel<<<1, 1, 0, st>>>(flag_up, flag_down, epoch);
    return after_launch();
}

#define LQCD_LAUNCH_SLAB_ARGS                                                                                          \
    const lqcd_ctx*, void*, const void*, const void*, const void*, const void*, const unsigned long long*,             \
        const unsigned long long*, unsigned long long, int, cudaStream_t, CbRange
#define LQCD_LAUNCH_FACES_ARGS                                                                                         \
    const lqcd_ctx*, const void*, void*, void*, unsigned long long*, unsigned long long*, unsigned long long, cudaStream_t

}  // namespace lqcd
