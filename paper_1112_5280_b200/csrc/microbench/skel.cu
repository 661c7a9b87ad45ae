// Memory skeleton of dslash_eo at 32^3x64 fp32/fp64 recon-12: same loads and stores, trivial arithmetic.
// MODE 0: all 72 loads issued up front.  MODE 1: hop k+1's loads depend on hop k's data (serialised like the real kernel).
#include <cstdio>
#include <cuda_runtime.h>

struct G { int Xh, Y, Z, T, Vh, sy, sz, st; size_t PS; };

template <typename W> __device__ __forceinline__ void addw(W& a, const W& b);
template <> __device__ __forceinline__ void addw<float4>(float4& a, const float4& b) { a.x += b.x; a.y += b.y; a.z += b.z; a.w += b.w; }
template <> __device__ __forceinline__ void addw<double2>(double2& a, const double2& b) { a.x += b.x; a.y += b.y; }
__device__ __forceinline__ int flag(const float4& a) { return a.x == 12345.f; }
__device__ __forceinline__ int flag(const double2& a) { return a.x == 12345.0; }

template <typename W, int NW, int Q, int MODE, int B, int LINKS, int NSPIN, int STORE, int TY, int TZ, int TT, int A>
__global__ void __launch_bounds__(B) skel(W* __restrict__ out, const W* __restrict__ gauge, const W* __restrict__ in, G g, int p) {
    int xh, y, z, t;
    {
        // block = tile of Xh x TY x TZ x TT sites (B == Xh*TY*TZ*TT); tiles ordered y fastest
        unsigned w = threadIdx.x; xh = w % g.Xh; w /= g.Xh; int yl = w % TY; w /= TY; int zl = w % TZ; int tl = w / TZ;
        unsigned b = blockIdx.x; int ty = b % (g.Y / TY); b /= (g.Y / TY); int tz = b % (g.Z / TZ); int tt = b / (g.Z / TZ);
        y = ty * TY + yl; z = tz * TZ + zl; t = tt * TT + tl;
    }
    const int cb = xh + g.Xh * (y + g.Y * (z + g.Z * t));
    int xo = (y + z + t + p) & 1;
    int nb[8];
    nb[0] = xo ? (xh == g.Xh - 1 ? cb - (g.Xh - 1) : cb + 1) : cb;
    nb[1] = xo ? cb : (xh == 0 ? cb + (g.Xh - 1) : cb - 1);
    nb[2] = y == g.Y - 1 ? cb - (g.Y - 1) * g.sy : cb + g.sy;
    nb[3] = y == 0 ? cb + (g.Y - 1) * g.sy : cb - g.sy;
    nb[4] = z == g.Z - 1 ? cb - (g.Z - 1) * g.sz : cb + g.sz;
    nb[5] = z == 0 ? cb + (g.Z - 1) * g.sz : cb - g.sz;
    nb[6] = t == g.T - 1 ? cb - (g.T - 1) * g.st : cb + g.st;
    nb[7] = t == 0 ? cb + (g.T - 1) * g.st : cb - g.st;
    W acc[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i) acc[i] = W{};
    int dep = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int mu = k / 2, fwd = !(k & 1);
        const int li = (fwd ? cb : nb[k]) + dep, si = nb[k] + dep;
        const size_t lstride = A ? 32 : g.PS, sstride = A ? 32 : g.PS;
        const W* lp = A == 2 ? gauge + ((size_t)(p * (g.Vh / 32) + (cb >> 5)) * 8 + k) * NW * 32 + (cb & 31) + dep
                    : A ? gauge + ((size_t)((fwd ? p : 1 - p) * (g.Vh / 32) + (li >> 5)) * 4 + mu) * NW * 32 + (li & 31)
                        : gauge + (size_t)(((fwd ? p : 1 - p) * 4 + mu) * NW) * g.PS + li;
        const W* sp = A ? in + (size_t)(si >> 5) * Q * 32 + (si & 31) : in + si;
        W l[NW], s[Q];
#pragma unroll
        for (int w = 0; w < NW; ++w) l[w] = LINKS ? __ldcs(lp + (size_t)w * lstride) : W{};
#pragma unroll
        for (int i = 0; i < Q; ++i) s[i] = (k < NSPIN) ? __ldg(sp + (size_t)i * sstride) : W{};
#pragma unroll
        for (int i = 0; i < Q; ++i) { addw(acc[i], s[i]); addw(acc[i], l[i % NW]); }
        if (MODE == 1) dep = flag(acc[0]);  // never 1, but the compiler cannot know
    }
#pragma unroll
    for (int i = 0; i < Q; ++i) if (STORE || flag(acc[i])) out[A ? (size_t)(cb >> 5) * Q * 32 + i * 32 + (cb & 31) : (size_t)i * g.PS + cb] = acc[i];
}

template <typename W, int NW, int Q, int MODE, int B, int LINKS, int NSPIN, int STORE, int TY, int TZ, int TT, int A>
void run(const char* name, size_t pad) {
    G g{16, 32, 32, 64, 16 * 32 * 32 * 64, 16, 16 * 32, 16 * 32 * 32, 0};
    g.PS = (size_t)g.Vh + pad;
    const int NBUF = 4;
    W *gauge, *in[NBUF], *out[NBUF];
    size_t gb = (size_t)(A == 2 ? 16 : 8) * NW * g.PS * sizeof(W), sb = (size_t)Q * g.PS * sizeof(W);
    cudaMalloc(&gauge, gb); cudaMemset(gauge, 0, gb);
    for (int i = 0; i < NBUF; ++i) { cudaMalloc(&in[i], sb); cudaMalloc(&out[i], sb); cudaMemset(in[i], 0, sb); }
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int N = 200;
    for (int i = 0; i < 20; ++i) skel<W, NW, Q, MODE, B, LINKS, NSPIN, STORE, TY, TZ, TT, A><<<g.Vh / B, B>>>(out[i % NBUF], gauge, in[i % NBUF], g, i & 1);
    cudaEventRecord(e0);
    for (int i = 0; i < N; ++i) skel<W, NW, Q, MODE, B, LINKS, NSPIN, STORE, TY, TZ, TT, A><<<g.Vh / B, B>>>(out[i % NBUF], gauge, in[i % NBUF], g, i & 1);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    double bytes = (double)(8 * NW * LINKS + (NSPIN ? Q : 0) + Q * STORE) * 16 * g.Vh;
    printf("%s links %d nspin %d store %d tile %dx%dx%d aosoa %d block %3d: %8.2f us  %8.1f GB/s (%s)\n", name, LINKS, NSPIN, STORE, TY, TZ, TT, A, B, ms / N * 1e3, bytes / (ms / N * 1e-3) / 1e9, cudaGetErrorString(cudaGetLastError()));
    cudaFree(gauge); for (int i = 0; i < NBUF; ++i) { cudaFree(in[i]); cudaFree(out[i]); }
}

int main() {
    for (int rep = 0; rep < 2; ++rep) {
        run<float4, 3, 6, 1, 64, 1, 8, 1, 4, 1, 1, 1>("fp32", 0);
        run<float4, 3, 6, 1, 64, 1, 8, 1, 4, 1, 1, 2>("fp32", 0);
        run<float4, 3, 6, 1, 128, 1, 8, 1, 8, 1, 1, 2>("fp32", 0);
        run<float4, 3, 6, 0, 64, 1, 8, 1, 4, 1, 1, 2>("fp32m0", 0);
        run<double2, 6, 12, 1, 64, 1, 8, 1, 4, 1, 1, 1>("fp64", 0);
        run<double2, 6, 12, 1, 64, 1, 8, 1, 4, 1, 1, 2>("fp64", 0);
        run<double2, 6, 12, 1, 128, 1, 8, 1, 8, 1, 1, 2>("fp64", 0);
        run<double2, 6, 12, 0, 64, 1, 8, 1, 4, 1, 1, 2>("fp64m0", 0);
    }
    return 0;
}
