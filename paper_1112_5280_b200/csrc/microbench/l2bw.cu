// Microbenchmark: L2-hit read bandwidth (working set fits L2) and mixed L2-hit + DRAM-stream traffic.
#include <cstdio>
#include <cuda_runtime.h>
// each thread: S loads from the DRAM-streamed buffer (unique), H loads from a small L2-resident buffer
template <int S, int H, int B>
__global__ void __launch_bounds__(B) rd(const float4* __restrict__ big, const float4* __restrict__ small_, float4* __restrict__ out,
                                         size_t stream_words, size_t small_words) {
    float4 acc = make_float4(0, 0, 0, 0);
    const size_t i = (size_t)blockIdx.x * B + threadIdx.x;
    float4 v[S + H + 1];
#pragma unroll
    for (int s = 0; s < S; ++s) v[s] = __ldcs(big + s * stream_words + i);
#pragma unroll
    for (int h = 0; h < H; ++h) v[S + h] = __ldcg(small_ + (i + (size_t)h * 4099 * B) % small_words);  // .cg: L2 only, no L1
#pragma unroll
    for (int s = 0; s < S + H; ++s) { acc.x += v[s].x; acc.y += v[s].y; acc.z += v[s].z; acc.w += v[s].w; }
    if (acc.x == 123.456f) out[i] = acc;
}
template <int S, int H, int B>
void run(const float4* big, const float4* small_, float4* out, size_t big_bytes, size_t small_bytes, size_t nthreads) {
    size_t sw = S ? big_bytes / 16 / S : 0;
    if (S) nthreads = sw;
    int nblk = (int)(nthreads / B);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int i = 0; i < 5; ++i) rd<S, H, B><<<nblk, B>>>(big, small_, out, sw, small_bytes / 16);
    cudaEventRecord(e0);
    const int N = 50;
    for (int i = 0; i < N; ++i) rd<S, H, B><<<nblk, B>>>(big, small_, out, sw, small_bytes / 16);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    double t = ms * 1e-3 / N;
    printf("S=%2d H=%2d B=%3d: dram %8.1f GB/s  l2hit %8.1f GB/s  total L2->SM %8.1f GB/s (%s)\n", S, H, B,
           (double)nthreads * S * 16 / t / 1e9, (double)nthreads * H * 16 / t / 1e9, (double)nthreads * (S + H) * 16 / t / 1e9,
           cudaGetErrorString(cudaGetLastError()));
}
int main() {
    size_t bytes = (size_t)1536 << 20, small_bytes = (size_t)24 << 20;
    float4 *in, *out, *sm; cudaMalloc(&in, bytes); cudaMalloc(&out, bytes); cudaMalloc(&sm, small_bytes);
    cudaMemset(in, 0, bytes); cudaMemset(sm, 0, small_bytes);
    size_t nthr = (size_t)16 << 20;
    for (int rep = 0; rep < 2; ++rep) {
        run<0, 8, 128>(in, sm, out, bytes, small_bytes, nthr);
        run<0, 16, 128>(in, sm, out, bytes, small_bytes, nthr);
        run<0, 32, 128>(in, sm, out, bytes, small_bytes, nthr);
        run<8, 0, 128>(in, sm, out, bytes, small_bytes, nthr);
        run<8, 2, 128>(in, sm, out, bytes, small_bytes, nthr);
        run<8, 4, 128>(in, sm, out, bytes, small_bytes, nthr);
        run<8, 8, 128>(in, sm, out, bytes, small_bytes, nthr);
        run<8, 16, 128>(in, sm, out, bytes, small_bytes, nthr);
    }
    return 0;
}
