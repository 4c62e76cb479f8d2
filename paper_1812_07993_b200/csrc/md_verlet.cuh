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

// flags: rebuild request, list overflow, position-buffer parity, velocity/id-buffer parity, rebuild count, escape
// The rebuild request rotates over three slots (step % 3): a slot is cleared one barrier before the phase that
// may set it and read one barrier after, so no block can see a later step's request (which would desynchronise
// the grid barriers).
enum { VF_REQ0 = 0, VF_OVERFLOW = 3, VF_CUR = 4, VF_CURV = 5, VF_NREBUILD = 6, VF_ESCAPE = 7, VF_COUNT = 8 };

template <typename T>
struct Verlet {
    // st[c].r: positions, double-buffered every step (nv vapor entries, then nw wall entries in cell order,
    // static); st[cv].{vx,vy,vz,id}: owner-only data, swapped only by the rebuild's scatter
    State<T> st[2];
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
// force: compute f from the list (else use the stored f(t));  kick: complete the current step (F3);
// drift: start the next step (F2).
template <typename T>
__device__ __forceinline__ void phase_step(const Params<T>& p, const Verlet<T>& v, int c, int cv, bool force,
                                           bool kick, bool drift, int req, int gtid, int gthreads)
{
    const Vec4<T>* __restrict__ rcur = v.st[c].r;
    Vec4<T>* __restrict__ rnew = v.st[c ^ 1].r;
    const State<T>& s = v.st[cv];
    const int g = gtid & (VL_G - 1);
    const int ngroups = gthreads / VL_G;
    for (int i0 = gtid / VL_G; i0 < ((p.nv + 3) & ~3); i0 += ngroups) {     // whole warps stay in the loop together
        const int i = min(i0, p.nv - 1);
        const Vec4<T> ri = rcur[i];
        T fx, fy, fz;
        if (force) {
            Acc<T, false> av, aw;
            list_force<T, false>(p, v, rcur, i, g, ri, av, aw);
            fx = group_sum(av.fx + aw.fx);
            fy = group_sum(av.fy + aw.fy);
            fz = group_sum(av.fz + aw.fz);
        } else {
            fx = v.f.fx[i]; fy = v.f.fy[i]; fz = v.f.fz[i];
        }
        if (g != 0 || i0 >= p.nv) continue;
        T vx = s.vx[i], vy = s.vy[i], vz = s.vz[i];
        if (force) { v.f.fx[i] = fx; v.f.fy[i] = fy; v.f.fz[i] = fz; }
        if (kick) {                                    // F3: v(t) = v(t - dt/2) + (dt/2m) f(t)
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
            if (rn.w > v.half_skin) v.flags[VF_REQ0 + req] = 1;
            rnew[i] = rn;
        }
        if (kick || drift) { s.vx[i] = vx; s.vy[i] = vy; s.vz[i] = vz; }
    }
}

// ---- rebuild phases (a2 inside the persistent kernel) -------------------------------------------
// R1: wrap periodic coordinates, cell id, count atomic -> slot.
template <typename T>
__device__ __forceinline__ void phase_bin(const Params<T>& p, const Verlet<T>& v, int c, int gtid, int gthreads)
{
    Vec4<T>* r = v.st[c].r;
    for (int i = gtid; i < p.nv; i += gthreads) {
        Vec4<T> ri = r[i];
        T dummy = T(0);
        int* err = v.flags + VF_ESCAPE;
        if (p.bc[0] == BC_PERIODIC) boundary(ri.x, dummy, p.L[0], BC_PERIODIC, err);
        if (p.bc[1] == BC_PERIODIC) boundary(ri.y, dummy, p.L[1], BC_PERIODIC, err);
        if (p.bc[2] == BC_PERIODIC) boundary(ri.z, dummy, p.L[2], BC_PERIODIC, err);
        ri.w = T(0);
        r[i] = ri;
        int cx, cy, cz;
        const int ci = cell_index(p, ri.x, ri.y, ri.z, cx, cy, cz);
        v.cell[i] = ci;
        v.slot[i] = atomicAdd(&v.count[ci], 1);
    }
}

// R2a / R2b: exclusive scan of the counts, tiles strided over the blocks (same arithmetic as
// k_scan_reduce / k_scan_apply).  blockDim.x must equal SCAN_THREADS.
__device__ __forceinline__ void phase_scan_reduce(const int* __restrict__ count, int n, int* __restrict__ tile_sum)
{
    __shared__ int ws[SCAN_THREADS / 32];
    const int tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
    for (int t = blockIdx.x; t < tiles; t += gridDim.x) {
        const int base = t * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
        int s = 0;
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k)
            if (base + k < n) s += count[base + k];
        s = warp_sum(s);
        __syncthreads();
        if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
        __syncthreads();
        if (threadIdx.x == 0) {
            int a = 0;
            for (int k = 0; k < SCAN_THREADS / 32; ++k) a += ws[k];
            tile_sum[t] = a;
        }
    }
}

__device__ __forceinline__ void phase_scan_apply(int* __restrict__ count, int n, const int* __restrict__ tile_sum,
                                                 int* __restrict__ start)
{
    __shared__ int ws[SCAN_THREADS / 32];
    __shared__ int s_off;
    const int tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
    for (int t = blockIdx.x; t < tiles; t += gridDim.x) {
        int off = 0;
        for (int k = threadIdx.x; k < t; k += SCAN_THREADS) off += tile_sum[k];
        off = warp_sum(off);
        __syncthreads();
        if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = off;
        __syncthreads();
        if (threadIdx.x == 0) {
            int a = 0;
            for (int k = 0; k < SCAN_THREADS / 32; ++k) a += ws[k];
            s_off = a;
        }
        __syncthreads();
        off = s_off;
        const int base = t * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
        int val[SCAN_ITEMS];
        int s = 0;
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) {
            val[k] = base + k < n ? count[base + k] : 0;
            s += val[k];
        }
        const int incl = warp_incl_scan(s);
        __syncthreads();
        if ((threadIdx.x & 31) == 31) ws[threadIdx.x >> 5] = incl;
        __syncthreads();
        int wofs = 0;
        for (int k = 0; k < (int)(threadIdx.x >> 5); ++k) wofs += ws[k];
        int run = off + wofs + incl - s;
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; ++k) {
            if (base + k < n) { start[base + k] = run; count[base + k] = 0; }
            run += val[k];
        }
        if (base <= n - 1 && n - 1 < base + SCAN_ITEMS) start[n] = run;
    }
}

// R3: scatter into cell order: positions c -> c^1, velocities / ids cv -> cv^1.
template <typename T>
__device__ __forceinline__ void phase_scatter(const Params<T>& p, const Verlet<T>& v, int c, int cv, int gtid,
                                              int gthreads)
{
    const State<T>& a = v.st[cv];
    const State<T>& b = v.st[cv ^ 1];
    const Vec4<T>* __restrict__ ra = v.st[c].r;
    Vec4<T>* __restrict__ rb = v.st[c ^ 1].r;
    for (int i = gtid; i < p.nv; i += gthreads) {
        const int d = v.start[v.cell[i]] + v.slot[i];
        rb[d] = ra[i];
        b.vx[d] = a.vx[i]; b.vy[d] = a.vy[i]; b.vz[d] = a.vz[i];
        b.id[d] = a.id[i];
    }
}

// R4: neighbour list from the cell list (a3's cell traversal, cached): every j within r_c + skin of i,
// vapor (j < nv) or wall (j = nv + k).  One thread per particle walks its 3^(d-1) cell rows; each row is
// one contiguous range of the cell-ordered arrays.  Positions are wrapped here, so distances fold.
template <typename T>
__device__ __forceinline__ int list_range(const Params<T>& p, const Vec4<T>* __restrict__ r, int jb, int je, int skip,
                                          const Vec4<T>& ri, T rl2, int* __restrict__ lst, int n)
{
    const bool px = p.bc[0] == BC_PERIODIC, py = p.bc[1] == BC_PERIODIC, pz = p.bc[2] == BC_PERIODIC;
    for (int j = jb; j < je; ++j) {
        if (j == skip) continue;
        const Vec4<T> rj = r[j];
        const T dx = px ? fold(ri.x, rj.x, p.L[0], T(0.5) * p.L[0]) : ri.x - rj.x;
        const T dy = py ? fold(ri.y, rj.y, p.L[1], T(0.5) * p.L[1]) : ri.y - rj.y;
        const T dz = pz ? fold(ri.z, rj.z, p.L[2], T(0.5) * p.L[2]) : ri.z - rj.z;
        const T r2 = fma_(dz, dz, fma_(dy, dy, dx * dx));
        if (r2 < rl2) {
            if (n < VL_MAXN) lst[n] = j;
            ++n;
        }
    }
    return n;
}

template <typename T, int ROWS>
__device__ __forceinline__ void phase_build(const Params<T>& p, const Verlet<T>& v, int c, int gtid, int gthreads)
{
    const Vec4<T>* __restrict__ r = v.st[c].r;
    const int nx = p.nc[0], ny = p.nc[1], nz = p.nc[2];
    for (int i = gtid; i < p.nv; i += gthreads) {
        const Vec4<T> ri = r[i];
        int cx, cy, cz;
        const int ci = cell_index(p, ri.x, ri.y, ri.z, cx, cy, cz);
        int* __restrict__ lst = v.nbr + (size_t)i * VL_MAXN;
        const bool do_wall = p.nw > 0 && v.wnear[ci];
        const int x0 = max(cx - 1, 0), x1 = min(cx + 1, nx - 1);
        int xw = -1;
        if (p.bc[0] == BC_PERIODIC) { if (cx == 0) xw = nx - 1; else if (cx == nx - 1) xw = 0; }
        int n = 0;
        for (int row = 0; row < ROWS; ++row) {
            int qy = cy + row % 3 - 1, qz = cz + (ROWS == 9 ? row / 3 - 1 : 0);
            if (qz < 0) { if (p.bc[2] != BC_PERIODIC) continue; qz += nz; }
            else if (qz >= nz) { if (p.bc[2] != BC_PERIODIC) continue; qz -= nz; }
            if (qy < 0) { if (p.bc[1] != BC_PERIODIC) continue; qy += ny; }
            else if (qy >= ny) { if (p.bc[1] != BC_PERIODIC) continue; qy -= ny; }
            const int rowc = (qz * ny + qy) * nx;
            n = list_range<T>(p, r, v.start[rowc + x0], v.start[rowc + x1 + 1], i, ri, v.rl2, lst, n);
            if (xw >= 0) n = list_range<T>(p, r, v.start[rowc + xw], v.start[rowc + xw + 1], i, ri, v.rl2, lst, n);
            if (do_wall) {
                n = list_range<T>(p, r, p.nv + v.wstart[rowc + x0], p.nv + v.wstart[rowc + x1 + 1], -1, ri, v.rl2, lst, n);
                if (xw >= 0)
                    n = list_range<T>(p, r, p.nv + v.wstart[rowc + xw], p.nv + v.wstart[rowc + xw + 1], -1, ri, v.rl2,
                                      lst, n);
            }
        }
        v.ncnt[i] = min(n, VL_MAXN);
        if (n > VL_MAXN) v.flags[VF_OVERFLOW] = 1;
    }
}

// ---- the persistent time loop ---------------------------------------------------------------------
// md_step(n): phase(stored f; kick + drift), then n - 1 fused phases (force; kick; kick + drift), then
// phase(force; kick): n + 1 phases and n grid barriers for n steps, plus 5 barriers per rebuild.
// force_rebuild (md_create): bin + build the list first, then evaluate f(0).
template <typename T, int ROWS>
__global__ void __launch_bounds__(VL_THREADS, 2) k_md_run(Params<T> p, Verlet<T> v, long long n_steps, int force_rebuild)
{
    cg::grid_group grid = cg::this_grid();
    const int gtid = blockIdx.x * blockDim.x + threadIdx.x;
    const int gthreads = gridDim.x * blockDim.x;
    int c = v.flags[VF_CUR], cv = v.flags[VF_CURV];
    bool rebuild = force_rebuild != 0;
    for (long long s = 0;; ++s) {
        if (rebuild) {
            phase_bin<T>(p, v, c, gtid, gthreads);
            grid.sync();
            phase_scan_reduce(v.count, p.ncell, v.tile_sum);
            grid.sync();
            phase_scan_apply(v.count, p.ncell, v.tile_sum, v.start);
            grid.sync();
            phase_scatter<T>(p, v, c, cv, gtid, gthreads);
            grid.sync();
            c ^= 1; cv ^= 1;
            phase_build<T, ROWS>(p, v, c, gtid, gthreads);
            if (gtid == 0) v.flags[VF_NREBUILD] += 1;
            grid.sync();
        }
        if (s == n_steps) break;
        const int req = (int)(s % 3);
        if (gtid == 0) v.flags[VF_REQ0 + (req + 1) % 3] = 0;      // slot of step s + 1
        phase_step<T>(p, v, c, cv, s > 0, s > 0, true, req, gtid, gthreads);
        grid.sync();
        c ^= 1;
        rebuild = *(volatile int*)(v.flags + VF_REQ0 + req) != 0;
    }
    if (n_steps > 0 || force_rebuild) phase_step<T>(p, v, c, cv, true, n_steps > 0, false, 0, gtid, gthreads);
    if (gtid == 0) { v.flags[VF_CUR] = c; v.flags[VF_CURV] = cv; }
}

// a5 energy pass over the neighbour list (ordinary launch; the host passes the buffer parities).
template <typename T>
__global__ void __launch_bounds__(VL_THREADS) k_verlet_energy(Params<T> p, Verlet<T> v, int c, EnergyOut eo)
{
    const int gtid = blockIdx.x * blockDim.x + threadIdx.x;
    const int g = gtid & (VL_G - 1);
    const int i0 = gtid / VL_G;
    const int i = min(i0, p.nv - 1);
    const Vec4<T>* __restrict__ r = v.st[c].r;
    const Vec4<T> ri = r[i];
    Acc<T, true> av, aw;
    list_force<T, true>(p, v, r, i, g, ri, av, aw);
    const double uv = group_sum(av.u), uw = group_sum(aw.u), wv = group_sum(av.w), ww = group_sum(aw.w);
    const int cvv = group_sum(av.c), cvw = group_sum(aw.c);
    if (g != 0 || i0 >= p.nv) return;
    eo.pe[i] = 0.5 * uv + uw;
    eo.pew[i] = uw;
    eo.vir[i] = 0.5 * wv + ww;
    eo.cvv[i] = cvv;
    eo.cvw[i] = cvw;
}

} // namespace md

namespace md {
// out[id[i]][0..dim) = r[i].xyz with periodic coordinates wrapped into [0, L) (the persistent kernel
// leaves them unwrapped between rebuilds).
template <typename T>
__global__ void k_export_pos_wrapped(Params<T> p, int dim, const int* __restrict__ id, const Vec4<T>* __restrict__ r,
                                     double* __restrict__ out)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.nv) return;
    Vec4<T> v = r[i];
    T dummy = T(0);
    int err = 0;
    if (p.bc[0] == BC_PERIODIC) boundary(v.x, dummy, p.L[0], BC_PERIODIC, &err);
    if (p.bc[1] == BC_PERIODIC) boundary(v.y, dummy, p.L[1], BC_PERIODIC, &err);
    if (p.bc[2] == BC_PERIODIC) boundary(v.z, dummy, p.L[2], BC_PERIODIC, &err);
    size_t o = (size_t)id[i] * dim;
    out[o] = (double)v.x;
    out[o + 1] = (double)v.y;
    if (dim == 3) out[o + 2] = (double)v.z;
}
} // namespace md
