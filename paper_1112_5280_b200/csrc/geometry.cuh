// geometry.cuh -- lattice geometry, checkerboard index maps and neighbour indexing (step K1).
//
// Conventions (the paper only says
// "even-odd preconditioning", and that NT, NS are fixed parameters):
//   mu = 0,1,2,3 = x,y,z,t;  lex = x + X(y + Y(z + Z t));  parity p = (x+y+z+t) & 1;
//   checkerboard index cb = lex >> 1 = xh + Xh(y + Y(z + Z t)),  xh = x >> 1,  Xh = X/2.
#pragma once
#include <cuda_runtime.h>

namespace lqcd {

struct Geom {
    int X, Y, Z, T;  // extents
    int Xh;          // X / 2
    int Vh;          // X*Y*Z*T / 2 (sites per parity)
    int ntiles;      // ceil(Vh / 32): 32-site tiles per parity in the native layout (fields.cuh)
    int sy, sz, st;  // cb strides of y, z, t: Xh, Xh*Y, Xh*Y*Z
    int tcf, tcb;    // t whose forward / backward hop carries the boundary phase: T-1 / 0 on a whole lattice; a
                     // time slab (lqcd_set_time_slab) moves them to where the global boundary cuts it, or -1
    // division by the run-time extents Xh, Y, Z without a divide: n / d = (n * mul) >> shift for every n < 2^30
    // (set_fastdiv; checkerboard indices are below 2^30 by lqcd_create)
    unsigned mul_xh, mul_y, mul_z;
    int sh_xh, sh_y, sh_z;
};

// mul = ceil(2^shift / d), shift = 30 + l, l = ceil(log2 d).  With e = mul d - 2^shift in [0, d):
// n mul / 2^shift = n / d + n e / (d 2^shift), and the excess is below 1 / d for n < 2^30 (n e < 2^30 2^l = 2^shift), so the
// floor is floor(n / d).  mul <= 2^31 fits in 32 bits.  (Checked against integer division in tests/test_abi.py.)
inline void set_fastdiv(unsigned d, unsigned& mul, int& shift) {
    int l = 0;
    while ((1u << l) < d) ++l;
    shift = 30 + l;
    mul = (unsigned)((((unsigned long long)1 << shift) + d - 1) / d);
}
__host__ __device__ __forceinline__ unsigned fastdiv(unsigned n, unsigned mul, int shift) {
    return (unsigned)(((unsigned long long)n * mul) >> shift);
}

struct Site {
    int xh, y, z, t;
    int x_odd;  // x & 1
};

// cb index -> coordinates for a site of parity p (A.5 inverse map).
__device__ __forceinline__ Site decode_site(const Geom& g, int cb, int p) {
    Site s;
    unsigned r = (unsigned)cb;
    unsigned q = fastdiv(r, g.mul_xh, g.sh_xh);
    s.xh = (int)(r - q * (unsigned)g.Xh);
    r = q;
    q = fastdiv(r, g.mul_y, g.sh_y);
    s.y = (int)(r - q * (unsigned)g.Y);
    r = q;
    q = fastdiv(r, g.mul_z, g.sh_z);
    s.z = (int)(r - q * (unsigned)g.Z);
    s.t = (int)q;
    s.x_odd = (s.y + s.z + s.t + p) & 1;
    return s;
}

// Neighbour of site (cb, s) one step along MU in direction FWD (true: +mu) in the
// opposite-parity array; `cross` is set when the hop wraps around the lattice (K3b).
template <int MU, bool FWD>
__device__ __forceinline__ int neighbour(const Geom& g, int cb, const Site& s, bool& cross) {
    if (MU == 0) {
        if (FWD) {
            // x even: x+1 shares xh.  x odd: xh+1, wrapping at Xh.
            cross = s.x_odd && (s.xh == g.Xh - 1);
            return s.x_odd ? (cross ? cb - (g.Xh - 1) : cb + 1) : cb;
        } else {
            cross = !s.x_odd && (s.xh == 0);
            return s.x_odd ? cb : (cross ? cb + (g.Xh - 1) : cb - 1);
        }
    } else if (MU == 1) {
        if (FWD) {
            cross = (s.y == g.Y - 1);
            return cross ? cb - (g.Y - 1) * g.sy : cb + g.sy;
        } else {
            cross = (s.y == 0);
            return cross ? cb + (g.Y - 1) * g.sy : cb - g.sy;
        }
    } else if (MU == 2) {
        if (FWD) {
            cross = (s.z == g.Z - 1);
            return cross ? cb - (g.Z - 1) * g.sz : cb + g.sz;
        } else {
            cross = (s.z == 0);
            return cross ? cb + (g.Z - 1) * g.sz : cb - g.sz;
        }
    } else {
        // the wrap decides the address, tcf / tcb decide where the boundary phase sits (the two differ on a time slab)
        if (FWD) {
            cross = (s.t == g.tcf);
            return (s.t == g.T - 1) ? cb - (g.T - 1) * g.st : cb + g.st;
        } else {
            cross = (s.t == g.tcb);
            return (s.t == 0) ? cb + (g.T - 1) * g.st : cb - g.st;
        }
    }
}

// the neighbour of hop k = 2 mu + (backward ? 1 : 0), k known only at run time (the producer warps of pipe_kernel.cuh)
__device__ __forceinline__ int neighbour_rt(const Geom& g, int cb, const Site& s, int k) {
    bool c;
    switch (k) {
        case 0: return neighbour<0, true>(g, cb, s, c);
        case 1: return neighbour<0, false>(g, cb, s, c);
        case 2: return neighbour<1, true>(g, cb, s, c);
        case 3: return neighbour<1, false>(g, cb, s, c);
        case 4: return neighbour<2, true>(g, cb, s, c);
        case 5: return neighbour<2, false>(g, cb, s, c);
        case 6: return neighbour<3, true>(g, cb, s, c);
        default: return neighbour<3, false>(g, cb, s, c);
    }
}

// K1 for one site: all eight neighbours (hop k = 2 mu + (backward ? 1 : 0)) and the bit mask of boundary-crossing hops.
__device__ __forceinline__ void all_neighbours(const Geom& g, int cb, const Site& s, int nb[8], unsigned& crossmask) {
    bool c;
    crossmask = 0;
    nb[0] = neighbour<0, true>(g, cb, s, c);  crossmask |= (unsigned)c << 0;
    nb[1] = neighbour<0, false>(g, cb, s, c); crossmask |= (unsigned)c << 1;
    nb[2] = neighbour<1, true>(g, cb, s, c);  crossmask |= (unsigned)c << 2;
    nb[3] = neighbour<1, false>(g, cb, s, c); crossmask |= (unsigned)c << 3;
    nb[4] = neighbour<2, true>(g, cb, s, c);  crossmask |= (unsigned)c << 4;
    nb[5] = neighbour<2, false>(g, cb, s, c); crossmask |= (unsigned)c << 5;
    nb[6] = neighbour<3, true>(g, cb, s, c);  crossmask |= (unsigned)c << 6;
    nb[7] = neighbour<3, false>(g, cb, s, c); crossmask |= (unsigned)c << 7;
}

}  // namespace lqcd
