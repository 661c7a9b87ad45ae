// fields.cuh -- native field layout (step L0), 256-/128-bit loads and stores (L1, L2, L6), K2 recon.
//
// Native layout (include/lqcd.h): array of structures of arrays with
// warp-sized tiles.  Sites of one parity are numbered by their checkerboard index cb and grouped in
// tiles of TILE = 32 consecutive cb (one warp); ntiles = ceil(Vh / 32), the last tile is padded.
//   spinor: real r = 6 spin + 2 colour + reim in [0,24); W = 32/sizeof(R) reals per 32-byte word,
//           Q = 24 / W words; word q of site cb at word index ((cb / 32) * Q + q) * 32 + cb % 32.
//           A warp reads word q of its 32 sites as one 1 KB run (one 256-bit access per lane), and the Q
//           words of a tile are adjacent: one contiguous 3 KB (fp32) / 6 KB (fp64) block per warp-level gather.
//   links:  "gathered by output site": for the site cb of parity p, hop k = 2 mu + (backward ? 1 : 0)
//           holds U_mu(x) (k even) or U_mu(x - mu^) (k odd), first RECON reals r = 6 row + 2 col + reim,
//           in words of LW reals; word w at ((((p * ntiles + cb / 32) * 8 + k) * NW + w) * 32 + cb % 32.
//           All 8 links of a warp's sites are one contiguous block read front to back (12 KB fp32
//           recon-12); every link is stored twice (as the forward link of x and the backward link of
//           x + mu^), which costs capacity, not traffic: one application reads each copy it needs once.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>

namespace lqcd {

constexpr int TILE = 32;

__device__ __forceinline__ float fmar(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fmar(double a, double b, double c) { return fma(a, b, c); }

// Spinor word: 32 bytes, read and written with Blackwell's 256-bit global accesses (LDG.256 / STG.256,
// ld.global.v8.f32 / .v4.f64 on sm_100): half as many memory instructions per byte as 128-bit words.
struct __align__(32) float8_ { float v[8]; };
struct __align__(32) double4_ { double v[4]; };
template <typename R> struct Word;
template <> struct Word<float>  { using type = float8_;  static constexpr int W = 8; };
template <> struct Word<double> { using type = double4_; static constexpr int W = 4; };

// Link word: the largest of 32 / 16 / 8 bytes that divides the stored reals (fp32 12-real: 3 x 16 B; fp32 18-real:
// 9 x 8 B; fp64 12-real: 3 x 32 B; fp64 18-real: 9 x 16 B).
template <typename R, int RECON> struct LinkWord;
template <> struct LinkWord<float, 12>  { using type = float4;   static constexpr int LW = 4; };
template <> struct LinkWord<float, 18>  { using type = float2;   static constexpr int LW = 2; };
template <> struct LinkWord<double, 12> { using type = double4_; static constexpr int LW = 4; };
template <> struct LinkWord<double, 18> { using type = double2;  static constexpr int LW = 2; };
template <> struct LinkWord<float, 13>  { using type = float4;   static constexpr int LW = 4; };  // RECON_12H: unused (half links)
template <> struct LinkWord<float, 8>   { using type = float4;   static constexpr int LW = 4; };  // 8-real: 2 x 16 B
template <> struct LinkWord<double, 8>  { using type = double4_; static constexpr int LW = 4; };  // 8-real: 2 x 32 B

__device__ __forceinline__ void unpack(const float4& w, float* v)  { v[0] = w.x; v[1] = w.y; v[2] = w.z; v[3] = w.w; }
__device__ __forceinline__ void unpack(const float2& w, float* v)  { v[0] = w.x; v[1] = w.y; }
__device__ __forceinline__ void unpack(const double2& w, double* v) { v[0] = w.x; v[1] = w.y; }
__device__ __forceinline__ void unpack(const float8_& w, float* v) {
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = w.v[i];
}
__device__ __forceinline__ void unpack(const double4_& w, double* v) {
#pragma unroll
    for (int i = 0; i < 4; ++i) v[i] = w.v[i];
}

// Cache policy of the field accesses: plain read-only (.nc) gathers and default stores.  L2::evict_last on the spinor
// gathers, .cs / L1::no_allocate.L2::evict_first on the 256-bit link words and .cs stores were each measured within
// +-0.5 % of this and are not kept as switches.
#define LQCD_LD_SPINOR "ld.global.nc"
#define LQCD_ST_SPINOR "st.global"
__device__ __forceinline__ float8_ ldg256(const float8_* p) {
    float8_ w;
    asm(LQCD_LD_SPINOR ".v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
        : "=f"(w.v[0]), "=f"(w.v[1]), "=f"(w.v[2]), "=f"(w.v[3]), "=f"(w.v[4]), "=f"(w.v[5]), "=f"(w.v[6]), "=f"(w.v[7]) : "l"(p));
    return w;
}
__device__ __forceinline__ double4_ ldg256(const double4_* p) {
    double4_ w;
    asm(LQCD_LD_SPINOR ".v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(w.v[0]), "=d"(w.v[1]), "=d"(w.v[2]), "=d"(w.v[3]) : "l"(p));
    return w;
}
// 256-bit link words (fp64 12-real / 8-real storage): read exactly once per application
__device__ __forceinline__ double4_ ldg256_stream(const double4_* p) {
    double4_ w;
    asm("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(w.v[0]), "=d"(w.v[1]), "=d"(w.v[2]), "=d"(w.v[3]) : "l"(p));
    return w;
}
// Plain (coherent) 256-bit loads for operands the same kernel overwrites (the in-place BLAS-1 updates): .nc is only
// legal for locations that stay read-only for the whole kernel.
__device__ __forceinline__ float8_ ld256(const float8_* p) {
    float8_ w;
    asm volatile("ld.global.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=f"(w.v[0]), "=f"(w.v[1]), "=f"(w.v[2]), "=f"(w.v[3]), "=f"(w.v[4]), "=f"(w.v[5]), "=f"(w.v[6]), "=f"(w.v[7])
                 : "l"(p) : "memory");
    return w;
}
__device__ __forceinline__ double4_ ld256(const double4_* p) {
    double4_ w;
    asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(w.v[0]), "=d"(w.v[1]), "=d"(w.v[2]), "=d"(w.v[3]) : "l"(p) : "memory");
    return w;
}
__device__ __forceinline__ void stg256(float8_* p, const float* v) {
    asm volatile(LQCD_ST_SPINOR ".v8.f32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(p), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]),
                 "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7]) : "memory");
}
__device__ __forceinline__ void stg256(double4_* p, const double* v) {
    asm volatile(LQCD_ST_SPINOR ".v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(v[0]), "d"(v[1]), "d"(v[2]), "d"(v[3]) : "memory");
}

// word 0 of site cb in a native half spinor; word q is q * TILE words further on
template <typename R>
__host__ __device__ __forceinline__ size_t spinor_word0(int cb) {
    constexpr int Q = 24 / Word<R>::W;
    return (size_t)((unsigned)cb / TILE) * (Q * TILE) + ((unsigned)cb % TILE);
}

// word 0 of hop k's link of site cb (parity p); word w is w * TILE words further on
template <typename R, int RECON>
__host__ __device__ __forceinline__ size_t link_word0(int ntiles, int p, int cb, int k) {
    constexpr int NW = RECON / LinkWord<R, RECON>::LW;
    return ((size_t)(p * ntiles + (int)((unsigned)cb / TILE)) * 8 + k) * (NW * TILE) + ((unsigned)cb % TILE);
}

// Spinor loads go through the read-only path (ld.global.nc) with default caching: each input spinor is gathered
// by 8 output sites, and that reuse must come from L1/L2, not from DRAM.  Only for fields the kernel never writes.
template <typename R>
__device__ __forceinline__ void load_spinor(const R* __restrict__ base, int cb, R v[24]) {
    using Wd = typename Word<R>::type;
    constexpr int W = Word<R>::W, Q = 24 / W;
    const Wd* p = reinterpret_cast<const Wd*>(base) + spinor_word0<R>(cb);
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        Wd w = ldg256(p + q * TILE);
        unpack(w, v + q * W);
    }
}

// the same for a field the calling kernel also writes (x, r, p of the CG updates): coherent loads
template <typename R>
__device__ __forceinline__ void load_spinor_rw(const R* base, int cb, R v[24]) {
    using Wd = typename Word<R>::type;
    constexpr int W = Word<R>::W, Q = 24 / W;
    const Wd* p = reinterpret_cast<const Wd*>(base) + spinor_word0<R>(cb);
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        Wd w = ld256(p + q * TILE);
        unpack(w, v + q * W);
    }
}

template <typename R>
__device__ __forceinline__ void store_spinor(R* __restrict__ base, int cb, const R v[24]) {
    using Wd = typename Word<R>::type;
    constexpr int W = Word<R>::W, Q = 24 / W;
    Wd* p = reinterpret_cast<Wd*>(base) + spinor_word0<R>(cb);
#pragma unroll
    for (int q = 0; q < Q; ++q) stg256(p + q * TILE, v + q * W);
}

// Links are read exactly once per application: streaming loads (ld.global.cs, evict-first)
// so they do not push the spinor working set out of L2.
__device__ __forceinline__ float4  ld_stream(const float4* p)  { return __ldcs(p); }
__device__ __forceinline__ float2  ld_stream(const float2* p)  { return __ldcs(p); }
__device__ __forceinline__ double2 ld_stream(const double2* p) { return __ldcs(p); }
__device__ __forceinline__ double4_ ld_stream(const double4_* p) { return ldg256_stream(p); }

// Packed fp32 arithmetic (Blackwell FFMA2 / FMUL2 / FADD2: two fp32 operations per instruction on an aligned register
// pair).  A complex number is one pair (re low, im high).  The SASS operand modifiers make a complex multiply-add two
// instructions with no data movement: a scalar operand is broadcast to both lanes (.F32), a pair can be read swapped
// (.LO_HI), and FADD2 can negate one half (.NP), so a complex sum  sum_b u_b z_b  is  P = sum ur (zr, zi),
// Q = sum ui (zi, zr)  (two FFMA2 per term)  and  (P.x - Q.x, P.y + Q.y)  (one FADD2).
// Each lane is an IEEE operation; the real and the imaginary-unit parts of a complex sum are accumulated in two
// chains and combined at the end (FFMA2 can negate a whole operand, FADD2 also one half of it), so the rounding order
// differs from the scalar code in the last bit -- every fp32 kernel variant shares these routines.
#ifndef LQCD_FFMA2
#define LQCD_FFMA2 1
#endif
struct P2 { unsigned long long v; };
__device__ __forceinline__ P2 pk(float lo, float hi) { P2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void unpk(P2 p, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p.v)); }
__device__ __forceinline__ P2 fma2(P2 a, P2 b, P2 c) { P2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d.v) : "l"(a.v), "l"(b.v), "l"(c.v)); return d; }
__device__ __forceinline__ P2 mul2(P2 a, P2 b) { P2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
__device__ __forceinline__ P2 add2(P2 a, P2 b) { P2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
__device__ __forceinline__ P2 bc2(float s) { return pk(s, s); }
template <typename R> constexpr bool packed_f32 = LQCD_FFMA2 && sizeof(R) == 4;

// K2: rebuild row 2 of u[18] (row-major 3x3 complex, u[6 row + 2 col + reim]) as conj(row0 x row1);
// valid for det U = +1 ("RECONSTRUCT TWELVE").
template <typename R>
__device__ __forceinline__ void recon_row2(R u[18]) {
    // row2[c] = conj(r0[a] r1[b] - r0[b] r1[a]),  (a,b) = (c+1, c+2) mod 3
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int a = (c + 1) % 3, b = (c + 2) % 3;
        const R ar = u[2 * a], ai = u[2 * a + 1], br = u[2 * b], bi = u[2 * b + 1];
        const R cr = u[6 + 2 * b], ci = u[6 + 2 * b + 1], dr = u[6 + 2 * a], di = u[6 + 2 * a + 1];
        if constexpr (packed_f32<R>) {
            // t = a c - b d with (re, im) as one pair: P = ar (cr, ci) - br (dr, di), Q = ai (ci, cr) - bi (di, dr) (swapped
            // reads), t = (P.x - Q.x, P.y + Q.y); FFMA2 negates whole operands only, FADD2 also one half
            P2 pp = mul2(bc2(ar), pk(cr, ci));
            pp = fma2(bc2(-br), pk(dr, di), pp);
            P2 qq = mul2(bc2(ai), pk(ci, cr));
            qq = fma2(bc2(-bi), pk(di, dr), qq);
            float qx, qy, re2, im2;
            unpk(qq, qx, qy);
            unpk(add2(pp, pk(-qx, qy)), re2, im2);
            u[12 + 2 * c] = re2;
            u[12 + 2 * c + 1] = -im2;
            continue;
        }
        const R re = fmar(-br, dr, fmar(bi, di, fmar(-ai, ci, ar * cr)));
        const R im = fmar(-br, di, fmar(-bi, dr, fmar(ai, cr, ar * ci)));
        u[12 + 2 * c] = re;
        u[12 + 2 * c + 1] = -im;
    }
}

// 8-real storage (next row f4, ref. [3] at :139): with the rows of U called a, b, c the stored reals are
//   r = (Re a1, Im a1, Re a2, Im a2, Re b0, Im b0, arg(a0) / pi, arg(c0) / pi)
// and, with N2 = |a1|^2 + |a2|^2:  a0 = sqrt(1 - N2) e^{i pi r6},  c0 = sqrt(N2 - |b0|^2) e^{i pi r7},
//   b1 = -(a1 conj(a0) b0 + conj(a2 c0)) / N2,   b2 = (conj(a1 c0) - a2 conj(a0) b0) / N2,   c = conj(a x b).
// (rows orthonormal, det = 1; the 2 x 2 system for b1, b2 has determinant N2.)  Singular for N2 = 0, i.e. |U00| = 1:
// unit links cannot be stored this way (lqcd_gauge_recon8_margin reports how close a field comes).
// Scalar helpers of the decoder, written out so that no library slow path (denormal / overflow handling of the IEEE
// division and square root, the general range reduction of sincospi) enters the kernel: every argument is in a known
// range here (N2 in (0, 1], the phases in [-1, 1]).
//   fp32: the special-function unit (MUFU.RCP / RSQ / SIN / COS); sin/cos.approx are accurate to 2^-20.9 absolute on
//         [-pi, pi], which puts the rebuilt link at ~5e-7 of the stored one -- below the 1e-5 bar of fp32 runs
//   fp64: MUFU.RCP64H / RSQ64H seeds (20 bits) + two Newton steps; sin(pi r), cos(pi r) by their Taylor series on
//         |r| <= 1/4 after reducing to the nearest quarter turn (truncation < 1e-16)
__device__ __forceinline__ float rcp_(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float rsqrt_(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ void sincospi_(float x, float& s, float& c) {
    const float a = 3.14159265358979f * x;
    asm("sin.approx.ftz.f32 %0, %1;" : "=f"(s) : "f"(a));
    asm("cos.approx.ftz.f32 %0, %1;" : "=f"(c) : "f"(a));
}
__device__ __forceinline__ double rcp_(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    r = fma(fma(-x, r, 1.0), r, r);
    r = fma(fma(-x, r, 1.0), r, r);
    return r;
}
__device__ __forceinline__ double rsqrt_(double x) {
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        const double e = fma(-x * r, r, 1.0);           // 1 - x r^2
        r = fma(fma(0.375, e, 0.5) * e, r, r);          // r (1 + e/2 + 3 e^2/8): third order, 20 -> 60 -> 180 bits
    }
    return r;
}
__device__ __forceinline__ void sincospi_(double x, double& s, double& c) {
    const double k = rint(2.0 * x);                      // nearest quarter turn, k in {-2, ..., 2}
    const double r = fma(k, -0.5, x), r2 = r * r;        // |r| <= 1/4
    double ps = -2.1915353447830215827e-5;
    ps = fma(ps, r2, 4.6630280576761256442e-4);
    ps = fma(ps, r2, -7.3704309457143507773e-3);
    ps = fma(ps, r2, 8.2145886611128228799e-2);
    ps = fma(ps, r2, -5.9926452932079207689e-1);
    ps = fma(ps, r2, 2.5501640398773454439);
    ps = fma(ps, r2, -5.1677127800499700292);
    ps = fma(ps, r2, 3.1415926535897932385);
    ps *= r;
    double pc = 4.3030695870329470073e-6;
    pc = fma(pc, r2, -1.0463810492484570712e-4);
    pc = fma(pc, r2, 1.9295743094039230479e-3);
    pc = fma(pc, r2, -2.5806891390014060013e-2);
    pc = fma(pc, r2, 2.3533063035889320454e-1);
    pc = fma(pc, r2, -1.3352627688545894959);
    pc = fma(pc, r2, 4.0587121264167682182);
    pc = fma(pc, r2, -4.9348022005446793094);
    pc = fma(pc, r2, 1.0);
    // rotate by k quarter turns: (c, s) -> (c cos(k pi/2) - s sin(k pi/2), s cos(k pi/2) + c sin(k pi/2))
    const int q = (int)k & 3;
    const double sw_s = (q & 1) ? pc : ps, sw_c = (q & 1) ? ps : pc;
    s = (q & 2) ? -sw_s : sw_s;
    c = ((q + 1) & 2) ? -sw_c : sw_c;
}

template <typename R>
__device__ __forceinline__ void recon8(const R r[8], R u[18]) {
    const R a1r = r[0], a1i = r[1], a2r = r[2], a2i = r[3], b0r = r[4], b0i = r[5];
    const R N2 = fmar(a1r, a1r, fmar(a1i, a1i, fmar(a2r, a2r, a2i * a2i)));
    const R B2 = fmar(b0r, b0r, b0i * b0i);
    R s0, c0, s2, c2;
    sincospi_(r[6], s0, c0);
    sincospi_(r[7], s2, c2);
    // sqrt(t) = t rsqrt(t), t clamped away from 0 (then the product is 0 to rounding, as it should be)
    constexpr R tiny = sizeof(R) == 4 ? (R)1e-30 : (R)1e-290;
    const R ta = fmax((R)1 - N2, tiny), tc = fmax(N2 - B2, tiny);
    const R ma = ta * rsqrt_(ta), mc = tc * rsqrt_(tc);
    const R a0r = ma * c0, a0i = ma * s0, c0r = mc * c2, c0i = mc * s2;
    const R inv = rcp_(N2);
    // t = conj(a0) b0;  w = a2 c0;  v = a1 c0
    const R tr = fmar(a0r, b0r, a0i * b0i), ti = fmar(a0r, b0i, -a0i * b0r);
    const R wr = fmar(a2r, c0r, -a2i * c0i), wi = fmar(a2r, c0i, a2i * c0r);
    const R vr = fmar(a1r, c0r, -a1i * c0i), vi = fmar(a1r, c0i, a1i * c0r);
    // b1 = -(a1 t + conj(w)) / N2;  b2 = (conj(v) - a2 t) / N2
    const R b1r = -inv * (fmar(a1r, tr, -a1i * ti) + wr), b1i = -inv * (fmar(a1r, ti, a1i * tr) - wi);
    const R b2r = inv * (vr - fmar(a2r, tr, -a2i * ti)), b2i = inv * (-vi - fmar(a2r, ti, a2i * tr));
    u[0] = a0r; u[1] = a0i; u[2] = a1r; u[3] = a1i; u[4] = a2r; u[5] = a2i;
    u[6] = b0r; u[7] = b0i; u[8] = b1r; u[9] = b1i; u[10] = b2r; u[11] = b2i;
    recon_row2<R>(u);
}

// ---- 16-bit storage (next row f4; "RECONSTRUCT TWELVE [3]" and the half-precision storage of ref. [3],
// PAPER.md:89, :139): fields are stored as IEEE half, the arithmetic stays fp32 --------------------------------
//   half spinor: 24 halfs = 3 16-byte words per site, [tile][q 3][32] as above, holding v / n(x) with
//                n(x) = max_k |v_k(x)| (so every stored number is in [-1, 1] and the 11-bit significand is
//                relative to the site's largest component); the fp32 norms n(x) follow the words of all tiles:
//                float[32 ntiles] at byte offset 48 * 32 * ntiles.  52 bytes per site.
//   links:       12-real storage only, 3 8-byte words of 4 halfs, [p][tile][hop 8][w 3][32]; entries of an SU(3)
//                matrix are in [-1, 1] already.  24 bytes per link.
constexpr int HALF_Q = 3;  // 16-byte words per half-precision spinor

__host__ __device__ __forceinline__ size_t half_spinor_words(int ntiles) { return (size_t)HALF_Q * TILE * ntiles; }

__device__ __forceinline__ void unpack_h8(const uint4& w, float* v) {
    const __half2* h = reinterpret_cast<const __half2*>(&w);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float2 f = __half22float2(h[i]);
        v[2 * i] = f.x;
        v[2 * i + 1] = f.y;
    }
}

// v = the stored (normalised) components, n = the site norm: the spinor is n * v.  The dslash kernel never
// forms n * v: the hop is linear, so n rides on the accumulation factor of step K5.
__device__ __forceinline__ void load_spinor_h(const __half* __restrict__ base, int ntiles, int cb, float v[24], float& n) {
    const uint4* words = reinterpret_cast<const uint4*>(base);
    const uint4* p = words + (size_t)((unsigned)cb / TILE) * (HALF_Q * TILE) + ((unsigned)cb % TILE);
    n = __ldg(reinterpret_cast<const float*>(words + half_spinor_words(ntiles)) + cb);
#pragma unroll
    for (int q = 0; q < HALF_Q; ++q) {
        const uint4 w = __ldg(p + q * TILE);
        unpack_h8(w, v + 8 * q);
    }
}
// the same with coherent loads, for a field the calling kernel also writes (p of the CG update)
__device__ __forceinline__ void load_spinor_h_rw(const __half* base, int ntiles, int cb, float v[24], float& n) {
    const uint4* words = reinterpret_cast<const uint4*>(base);
    const uint4* p = words + (size_t)((unsigned)cb / TILE) * (HALF_Q * TILE) + ((unsigned)cb % TILE);
    asm volatile("ld.global.f32 %0, [%1];" : "=f"(n) : "l"(reinterpret_cast<const float*>(words + half_spinor_words(ntiles)) + cb) : "memory");
#pragma unroll
    for (int q = 0; q < HALF_Q; ++q) {
        uint4 w;
        asm volatile("ld.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(w.x), "=r"(w.y), "=r"(w.z), "=r"(w.w) : "l"(p + q * TILE) : "memory");
        unpack_h8(w, v + 8 * q);
    }
}

// the stored words themselves (for the mixed-precision projection of dslash_kernel.cuh) and the site norm
__device__ __forceinline__ void load_words_h(const __half* __restrict__ base, int ntiles, int cb, uint4 w[3], float& n) {
    const uint4* words = reinterpret_cast<const uint4*>(base);
    const uint4* p = words + (size_t)((unsigned)cb / TILE) * (HALF_Q * TILE) + ((unsigned)cb % TILE);
    n = __ldg(reinterpret_cast<const float*>(words + half_spinor_words(ntiles)) + cb);
#pragma unroll
    for (int q = 0; q < HALF_Q; ++q) w[q] = __ldg(p + q * TILE);
}

__device__ __forceinline__ void store_spinor_h(__half* __restrict__ base, int ntiles, int cb, const float v[24]) {
    uint4* words = reinterpret_cast<uint4*>(base);
    uint4* p = words + (size_t)((unsigned)cb / TILE) * (HALF_Q * TILE) + ((unsigned)cb % TILE);
    float n = 0.f;
#pragma unroll
    for (int k = 0; k < 24; ++k) n = fmaxf(n, fabsf(v[k]));
    const float inv = n > 0.f ? 1.f / n : 0.f;
#pragma unroll
    for (int q = 0; q < HALF_Q; ++q) {
        uint4 w;
        __half2* h = reinterpret_cast<__half2*>(&w);
#pragma unroll
        for (int i = 0; i < 4; ++i) h[i] = __floats2half2_rn(v[8 * q + 2 * i] * inv, v[8 * q + 2 * i + 1] * inv);
        p[q * TILE] = w;
    }
    reinterpret_cast<float*>(words + half_spinor_words(ntiles))[cb] = n;
}

// word 0 of hop k's link of site cb (parity p) in the half-precision link field, in 8-byte words
__host__ __device__ __forceinline__ size_t link_word0_h(int ntiles, int p, int cb, int k) {
    return ((size_t)(p * ntiles + (int)((unsigned)cb / TILE)) * 8 + k) * (3 * TILE) + ((unsigned)cb % TILE);
}

__device__ __forceinline__ void load_link_h(const uint2* __restrict__ site_links, int k, float u[18]) {
#pragma unroll
    for (int w = 0; w < 3; ++w) {
        const uint2 x = __ldcs(site_links + (k * 3 + w) * TILE);
        const __half2* h = reinterpret_cast<const __half2*>(&x);
        const float2 a = __half22float2(h[0]), b = __half22float2(h[1]);
        u[4 * w] = a.x; u[4 * w + 1] = a.y; u[4 * w + 2] = b.x; u[4 * w + 3] = b.y;
    }
    recon_row2<float>(u);
}

// Storage type S -> arithmetic type, and uniform field access for the kernels (ntiles is only used by half).
template <typename S> struct Compute { using type = S; };
template <> struct Compute<__half> { using type = float; };

// the spinor at cb is scale * v (scale = 1 for fp32 / fp64 storage)
template <typename S>
__device__ __forceinline__ void load_field(const S* __restrict__ base, int ntiles, int cb, typename Compute<S>::type v[24],
                                           typename Compute<S>::type& scale) {
    if constexpr (sizeof(S) == 2) {
        load_spinor_h(base, ntiles, cb, v, scale);
    } else {
        load_spinor<S>(base, cb, v);
        scale = 1;
    }
}
template <typename S>
__device__ __forceinline__ void store_field(S* __restrict__ base, int ntiles, int cb, const typename Compute<S>::type v[24]) {
    if constexpr (sizeof(S) == 2) store_spinor_h(base, ntiles, cb, v); else store_spinor<S>(base, cb, v);
}
// elements of S between the even and the odd half of a native full spinor
template <typename S>
__host__ __device__ __forceinline__ size_t half_stride(int ntiles) {
    return sizeof(S) == 2 ? (size_t)(24 + 2) * TILE * ntiles : (size_t)24 * TILE * ntiles;
}

// storage-type view of the link field
template <typename S, int RECON> struct LinkStore {
    using R = typename Compute<S>::type;
    using word = typename LinkWord<R, RECON>::type;
    static constexpr int R_PER_WORD = LinkWord<R, RECON>::LW;
    static __host__ __device__ __forceinline__ size_t word0(int ntiles, int p, int cb, int k) { return link_word0<R, RECON>(ntiles, p, cb, k); }
};
template <int RECON> struct LinkStore<__half, RECON> {
    using R = float;
    using word = uint2;
    static constexpr int R_PER_WORD = 4;
    static __host__ __device__ __forceinline__ size_t word0(int ntiles, int p, int cb, int k) { return link_word0_h(ntiles, p, cb, k); }
};
// fp32 spinors with the links stored as 12 halfs (lqcd_params.link_precision = 16): the link stream is 2/3 of
// the traffic, and a 2^-11 perturbation of the links is harmless for the inner solver of a defect correction
constexpr int RECON_12H = 13;
template <> struct LinkStore<float, RECON_12H> {
    using R = float;
    using word = uint2;
    static constexpr int R_PER_WORD = 4;
    static __host__ __device__ __forceinline__ size_t word0(int ntiles, int p, int cb, int k) { return link_word0_h(ntiles, p, cb, k); }
};
template <typename S, int RECON> constexpr bool half_links = sizeof(S) == 2 || RECON == RECON_12H;

// L1 + K2: link of hop k for the site whose hop-0 word-0 address is `site_links`.
template <typename R, int RECON>
__device__ __forceinline__ void load_link(const typename LinkWord<R, RECON>::type* __restrict__ site_links, int k, R u[18]) {
    using LWd = typename LinkWord<R, RECON>::type;
    constexpr int LW = LinkWord<R, RECON>::LW, NW = RECON / LW;
    if constexpr (RECON == 8) {
        R r[8];
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            LWd x = ld_stream(site_links + (k * NW + w) * TILE);
            unpack(x, r + w * LW);
        }
        recon8<R>(r, u);
    } else {
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            LWd x = ld_stream(site_links + (k * NW + w) * TILE);
            unpack(x, u + w * LW);
        }
        if constexpr (RECON == 12) recon_row2<R>(u);
    }
}

}  // namespace lqcd
