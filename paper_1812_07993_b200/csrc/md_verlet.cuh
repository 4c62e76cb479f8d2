// md_verlet.cuh -- persistent (cooperative) time-loop kernel: cell list -> Verlet list with skin.
//
// Why (profiles/r01_v2_cfg2.md): at N ~ 1e5 a time step is launch- and latency-bound.  A CUDA-graph
// step of 5 kernels costs 35 us where its arithmetic needs < 1 us, a never-taken conditional graph
// node costs ~7 us (measured), and walking 3^d cells per particle executes ~10x the useful
// instructions.  So the whole md_step(n) batch is ONE cooperative launch: every time step is one
// fused phase  [F1 forces from the cached neighbour list -> F3 half-kick -> F2 half-kick + drift]
// followed by one grid barrier, and the cell list (a2: count atomics, scan,
// scatter) plus the neighbour list are rebuilt inside the kernel only when some particle's path
// since the last rebuild exceeds skin/2 -- the list holds every pair within r_c + skin, so every
// pair within r_c is evaluated at every step: results are exact, identical to the brute-force
// definition up to summation order.
#pragma once
#include "md_kernels.cuh"

#include <cooperative_groups.h>

namespace md {
namespace cg = cooperative_groups;

constexpr int VL_THREADS = 256;
constexpr int VL_G = 8;        // lanes cooperating on one particle in the force phase
constexpr int VL_MAXN = 128;   // neighbour-list stride (entries per particle)

enum { VF_REBUILD = 0, VF_OVERFLOW = 1, VF_CUR = 2, VF_NREBUILD = 3, VF_ESCAPE = 4, VF_COUNT = 8 };

template <typename T>
struct Verlet {
    State<T> st[2];            // r holds nv vapor entries followed by nw wall entries (cell order, static)
    Force<T> f;
    int *nbr, *ncnt;           // [nv * VL_MAXN], [nv]; j >= nv means wall particle j - nv
    int *cell, *slot, *count, *start, *tile_sum;
    const int* wstart;         // walls: [ncell + 1] ranges into the wall tail
    const uint8_t* wnear;
    int* flags;                // VF_*
    T rl2, half_skin;          // (r_c + skin)^2, skin / 2
};

// d = a - b folded to the nearest image by comparison (|true d| < r_c + skin < L/2).  fp32: the shift
// goes on whichever particle sits at the top of the box so the difference stays exact.
__device__ __forceinline__ double fold(double a, double b, double L, double halfL)
{
    double d = a - b;
    if (d > halfL) d -= L;
    else if (d < -halfL) d += L;
    return d;
}
__device__ __forceinline__ float fold(float a, float b, float L, float halfL)
{
    float d = a - b;
    if (d > halfL) d = (a - L) - b;
    else if (d < -halfL) d = a - (b - L);
    return d;
}

template <typename V>
__device__ __forceinline__ V group_sum(V v)
{
#pragma unroll
    for (int o = VL_G / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---- one particle's force from its neighbour list, VL_G lanes ---------------------------------
template <typename T, bool ENERGY>
__device__ __forceinline__ void list_force(const Params<T>& p, const Verlet<T>& v, const Vec4<T>* __restrict__ r, int i,
                                           int g, const Vec4<T>& ri, Acc<T, ENERGY>& av, Acc<T, ENERGY>& aw)
{
    const int n = v.ncnt[i];
    const int* __restrict__ lst = v.nbr + (size_t)i * VL_MAXN;
    const bool px = p.bc[0] == BC_PERIODIC, py = p.bc[1] == BC_PERIODIC, pz = p.bc[2] == BC_PERIODIC;
    for (int k = g; k < n; k += VL_G) {
        const int j = lst[k];
        const Vec4<T> rj = r[j];
        T dx = px ? fold(ri.x, rj.x, p.L[0], T(0.5) * p.L[0]) : ri.x - rj.x;
        T dy = py ? fold(ri.y, rj.y, p.L[1], T(0.5) * p.L[1]) : ri.y - rj.y;
        T dz = pz ? fold(ri.z, rj.z, p.L[2], T(0.5) * p.L[2]) : ri.z - rj.z;
        if (j < p.nv) pair_term<T, ENERGY>(dx, dy, dz, p.rc2, p.sig2_vv, p.e24_vv, p.e4_vv, p.uc_vv, av);
        else pair_term<T, ENERGY>(dx, dy, dz, p.rc2, p.sig2_vw, p.e24_vw, p.e4_vw, p.uc_vw, aw);
    }
}

// ---- phase: [forces] -> [kick completing the step] -> [kick + drift of the next step] -----------
// FORCE: compute f from the list (else use the stored f(t));  DRIFT: start the next step.
template <typename T>
__device__ __forceinline__ void phase_step(const Params<T>& p, const Verlet<T>& v, int c, bool force, bool drift,
                                           int gtid, int gthreads)
{
    const State<T>& s = v.st[c];
    const State<T>& o = v.st[c ^ 1];
    const int g = gtid & (VL_G - 1);
    const int ngroups = gthreads / VL_G;
    for (int i0 = gtid / VL_G; i0 < ((p.nv + 3) & ~3); i0 += ngroups) {     // whole warps stay in the loop together
        const int i = min(i0, p.nv - 1);
        const Vec4<T> ri = s.r[i];
        T fx, fy, fz;
        if (force) {
            Acc<T, false> av, aw;
            list_force<T, false>(p, v, s.r, i, g, ri, av, aw);
            fx = group_sum(av.fx + aw.fx);
            fy = group_sum(av.fy + aw.fy);
            fz = group_sum(av.fz + aw.fz);
        } else {
            fx = v.f.fx[i]; fy = v.f.fy[i]; fz = v.f.fz[i];
        }
        if (g != 0 || i0 >= p.nv) continue;
        T vx = s.vx[i], vy = s.vy[i], vz = s.vz[i];
        if (force) {                                   // F3: v(t) = v(t - dt/2) + (dt/2m) f(t)
            v.f.fx[i] = fx; v.f.fy[i] = fy; v.f.fz[i] = fz;
            vx = vx + p.hk * fx; vy = vy + p.hk * fy; vz = vz + p.hk * fz;
        }
        if (drift) {                                   // F2: v(t + dt/2), r(t + dt)
            vx = vx + p.hk * fx; vy = vy + p.hk * fy; vz = vz + p.hk * fz;
            const T sx = p.dt * vx, sy = p.dt * vy, sz = p.dt * vz;
            Vec4<T> rn;
            rn.x = ri.x + sx; rn.y = ri.y + sy; rn.z = ri.z + sz;
            // periodic dimensions are left unwrapped until the next rebuild; reflection is immediate
            int* err = v.flags + VF_ESCAPE;
            if (p.bc[0] == BC_REFLECT) boundary(rn.x, vx, p.L[0], BC_REFLECT, err);
            if (p.bc[1] == BC_REFLECT) boundary(rn.y, vy, p.L[1], BC_REFLECT, err);
            if (p.bc[2] == BC_REFLECT) boundary(rn.z, vz, p.L[2], BC_REFLECT, err);
            rn.w = ri.w + sqrt(sx * sx + sy * sy + sz * sz);      // path length >= displacement
            if (rn.w > v.half_skin) v.flags[VF_REBUILD] = 1;
            o.r[i] = rn;
            o.vx[i] = vx; o.vy[i] = vy; o.vz[i] = vz;
        } else if (force) {
            s.vx[i] = vx; s.vy[i] = vy; s.vz[i] = vz;
        }
    }
}
