// Microbenchmark: read-bandwidth vs number of concurrent streams (each block reads 64x16 B = 1 KB from each of S streams).
#include <cstdio>
#include <cuda_runtime.h>
template <int S, int B>
__global__ void __launch_bounds__(B) rd(const float4* __restrict__ in, float4* __restrict__ out, size_t stream_words, int nblk) {
    float4 acc = make_float4(0, 0, 0, 0);
    const size_t i = (size_t)blockIdx.x * B + threadIdx.x;
    float4 v[S];
#pragma unroll
    for (int s = 0; s < S; ++s) v[s] = __ldcs(in + s * stream_words + i);
#pragma unroll
    for (int s = 0; s < S; ++s) { acc.x += v[s].x; acc.y += v[s].y; acc.z += v[s].z; acc.w += v[s].w; }
    if (acc.x == 123.456f) out[i] = acc;  // never true: keeps the loads alive
}
template <int S, int B>
void run(const float4* in, float4* out, size_t total_bytes) {
    size_t words = total_bytes / 16, sw = words / S;
    int nblk = (int)(sw / B);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int i = 0; i < 5; ++i) rd<S, B><<<nblk, B>>>(in, out, sw, nblk);
    cudaEventRecord(e0);
    const int N = 50;
    for (int i = 0; i < N; ++i) rd<S, B><<<nblk, B>>>(in, out, sw, nblk);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    printf("S=%2d B=%3d: %8.1f GB/s  (%s)\n", S, B, (double)sw * S * 16 * N / (ms * 1e-3) / 1e9, cudaGetErrorString(cudaGetLastError()));
}
int main() {
    size_t bytes = (size_t)1536 << 20;
    float4 *in, *out; cudaMalloc(&in, bytes); cudaMalloc(&out, bytes); cudaMemset(in, 0, bytes);
    for (int rep = 0; rep < 2; ++rep) {
        run<1, 64>(in, out, bytes); run<2, 64>(in, out, bytes); run<4, 64>(in, out, bytes); run<8, 64>(in, out, bytes);
        run<12, 64>(in, out, bytes); run<24, 64>(in, out, bytes); run<36, 64>(in, out, bytes);
        run<1, 256>(in, out, bytes); run<4, 256>(in, out, bytes); run<8, 256>(in, out, bytes); run<24, 256>(in, out, bytes);
        run<24, 32>(in, out, bytes); run<8, 32>(in, out, bytes);
    }
    return 0;
}
