// pm_pos.cuh -- device helpers shared by the kernels that turn the integrator state into sort keys:
// state coordinate (int64, 2^-XBITS cells, absolute and unwrapped) -> 32-bit record coordinate
// (cell << fbits | fraction, wrapped into the mesh) -> (tile, class) key of the cell sort (pm_bin.cu).
#pragma once
#include "pm_internal.cuh"

namespace pm {

struct PosGeom {
    unsigned long long M[3];  // N << fbits: period of the record coordinate
    long long qstep[3];       // lattice spacing in state units: (N << XBITS) / L
    int N[3], L[3], nt[3];
    int fbits;
    int pow2[3];              // N is a power of two
};

__device__ __forceinline__ unsigned int wrap_fixed(long long v, unsigned long long M, int pow2)
{
    if (pow2) return (unsigned int)((unsigned long long)v & (M - 1ull));
    long long m = (long long)M;
    long long r = v % m;
    if (r < 0) r += m;
    return (unsigned int)r;
}

// state coordinate -> record coordinate, rounded to nearest (a deterministic function of the state,
// so F(x) stays bit-reproducible in the reverse pass)
__device__ __forceinline__ unsigned int record_coord(const PosGeom &g, long long x, int d)
{
    const int sh = XBITS - g.fbits;
    long long v = (x + (1ll << (sh - 1))) >> sh;
    return wrap_fixed(v, g.M[d], g.pow2[d]);
}

__device__ __forceinline__ int key_of(const PosGeom &g, const unsigned int X[3])
{
    int c0 = (int)(X[0] >> g.fbits), c1 = (int)(X[1] >> g.fbits), c2 = (int)(X[2] >> g.fbits);
    int t0 = c0 / TX, t1 = c1 / TY, t2 = c2 / TZ;
    int e0 = min(t0 * TX + TX, g.N[0]) - 1, e1 = min(t1 * TY + TY, g.N[1]) - 1, e2 = min(t2 * TZ + TZ, g.N[2]) - 1;
    int cls = ((c0 == e0) << 2) | ((c1 == e1) << 1) | (int)(c2 == e2);
    return ((t0 * g.nt[1] + t1) * g.nt[2] + t2) * NCLS + cls;
}

// histogram increment, one atomic per distinct key among the converged lanes
__device__ __forceinline__ void hist_add(int *hist, int key)
{
    unsigned int act = __activemask();
    unsigned int peers = __match_any_sync(act, key);
    int lane = threadIdx.x & 31;
    if (lane == __ffs(peers) - 1) atomicAdd(hist + key, __popc(peers));
}

PosGeom make_pos_geom(const Geometry &g);

// fused kick / kick / drift applied by the gather kernels right after they have interpolated acc (and alpha)
// for a particle (eq. 16; eq. 49): p += rn(acc Ka); [p += rn(acc Kb);] [x += rn(p D)], each
// rounded separately so that the reverse pass mirrors the forward pass bit for bit (R14).
struct KickArgs {
    double Ka, Kb, Ds;        // scaled: K * 2^PBITS, D * 2^(XBITS - PBITS); 0 = skip
    float Kaf, Kbf, Df;       // plain factors for the adjoint variables
    long long *x, *p;         // state
    float *xi, *pi;           // adjoint variables (adjoint kernels only)
    int *hist;                // key histogram of the new positions (when Ds != 0)
    int enabled;              // 0: plain gather
    int store;                // also write acc (and alpha) to memory
};

}  // namespace pm
