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
};

struct Site {
    int xh, y, z, t;
    int x_odd;  // x & 1
};

// cb index -> coordinates for a site of parity p (A.5 inverse map).
__device__ __forceinline__ Site decode_site(const Geom& g, int cb, int p) {
    Site s;
    unsigned r = (unsigned)cb;
    unsigned q = r / (unsigned)g.Xh;
    s.xh = (int)(r - q * (unsigned)g.Xh);
    r = q;
    q = r / (unsigned)g.Y;
    s.y = (int)(r - q * (unsigned)g.Y);
    r = q;
    q = r / (unsigned)g.Z;
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

}  // namespace lqcd
