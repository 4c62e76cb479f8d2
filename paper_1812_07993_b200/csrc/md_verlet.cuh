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
constexpr int VL_MAXN = 128;   // neighbour-list stride (entries per particle)

// flags: rebuild request, list overflow, position-buffer parity, velocity/id-buffer parity, rebuild count, escape,
// particles with a long list at the last rebuild (demand), how many of them the idle blocks' lane groups took (capacity)
// The rebuild request rotates over three slots (step % 3): a slot is cleared one barrier before the phase that
// may set it and read one barrier after, so no block can see a later step's request (which would desynchronise
// the grid barriers).
enum { VF_REQ0 = 0, VF_OVERFLOW = 3, VF_CUR = 4, VF_CURV = 5, VF_NREBUILD = 6, VF_ESCAPE = 7, VF_NHEAVY = 8, VF_HCAP = 9, VF_COUNT = 10 };

template <typename T>
struct Verlet {
    // st[c].r: positions, double-buffered every step (nv vapor entries, then nw wall entries in cell order,
    // static); st[cv].{vx,vy,vz,id}: owner-only data, swapped only by the rebuild's scatter
    State<T> st[2];
    Force<T> f;
    int *nbr, *ncnt;           // nbr[k * stride + i], k < VL_MAXN; ncnt[nv]; j >= nv means wall particle j - nv
    size_t stride;             // >= nv
    int *cell, *slot, *count, *start, *tile_sum;
    const int* wstart;         // walls: [ncell + 1] ranges into the wall tail
    const uint8_t* wnear;
    int* flags;                // VF_*
    unsigned long long* bar;   // grid barrier arrival counter
    double* ksum;              // [3] kinetic-energy accumulators of the thermostat, rotating like the requests
    unsigned long long* dbg;   // optional per-warp step-phase ns (diagnostics), or nullptr
    unsigned long long* times; // [8] ns seen by thread 0: step phases, step barriers, rebuilds, final phase,
                               // rebuild split: bin, scan, scatter, list build (each with its barrier)
    T rl2, half_skin;          // (r_c + skin)^2, skin / 2
    int carry;                 // 0: reload own state every step (diagnostic A/B, MD_NO_CARRY)
    int heavy_t;               // particles whose list is longer than this are "heavy": in the step phase an 8-lane
                               // group shares one such list (indices in `cell`, ncnt words in `slot` -- both free
                               // between rebuilds; their number in flags[VF_NHEAVY])
};

// d = a - b folded to the nearest image by comparison (|true d| < r_c + skin < L/2).  fp32: the shift
// goes on whichever particle sits at the top of the box so the difference stays exact.
// fp64: |d| > L/2 is decided on the high word by the integer pipe (|d| is either < r_c + skin or > L - r_c - skin,
// never near L/2) and the shift is L with d's sign: 2 FP64 instructions instead of 5 (DADD, 2 DSETP, 2 predicated
// DADD) in a loop that is bound by the FP64 pipe (profiles/r01_heavy_groups.md); the result is bit-identical.
__device__ __forceinline__ double fold(double a, double b, double L, double halfL)
{
    double d = a - b;
    const int hi = __double2hiint(d);
    if ((hi & 0x7fffffff) > __double2hiint(halfL))
        d -= __hiloint2double(__double2hiint(L) | (hi & 0x80000000), __double2loint(L));
    return d;
}
__device__ __forceinline__ float fold(float a, float b, float L, float halfL)
{
    float d = a - b;
    if (d > halfL) d = (a - L) - b;
    else if (d < -halfL) d = a - (b - L);
    return d;
}

// Grid barrier of the cooperative launch (all blocks are co-resident).  One arrival atomic per block; the wait
// polls with relaxed loads and fences ONCE when released -- cooperative_groups' grid.sync() re-acquires (and so
// invalidates the SM's L1, CCTL.IVALL) on every poll, which also evicts the lines of the other block still
// computing on that SM (profiles/r01_v3_cfg2.md).  `bar` is zeroed by the host before every launch.
__device__ __forceinline__ void grid_barrier(unsigned long long* bar, unsigned long long& target)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        target += gridDim.x;
        __threadfence();                                   // release this block's writes
        atomicAdd(bar, 1ull);
        unsigned long long seen;
        do {
            asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(seen) : "l"(bar) : "memory");
        } while (seen < target);
        __threadfence();                                   // acquire: later loads see every block's writes
    }
    __syncthreads();
}

__device__ __forceinline__ unsigned long long now_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}

// ---- one particle's force from its neighbour list, one thread per particle ----------------------
// The list is stored transposed, nbr[k * stride + i], so a warp's loads of entry k are coalesced.
// ncnt[i] = list length | VL_FOLD if the particle sat in a cell on a periodic face when the list was
// built: only such particles can have a neighbour across the face, all others skip the image folding.
// Entries are consumed four at a time: four index loads, then four position loads, are in flight together.
constexpr int VL_FOLD = 1 << 30;
constexpr int VL_HEAVY = 1 << 29;      // list longer than Verlet::heavy_t (see phase_step)
constexpr int VL_NMASK = (1 << 16) - 1;
#ifndef MD_VL_GROUP
#define MD_VL_GROUP 4
#endif
constexpr int VL_GROUP = MD_VL_GROUP;   // lanes sharing one heavy particle's list

// 1 / x without the division's special-case branch: hardware seed (>= 20 bits) + two Newton steps.
__device__ __forceinline__ double rcp_fast(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
}
__device__ __forceinline__ float rcp_fast(float x) { return 1.0f / x; }

// |step| rounded UP for the path-length bound: the fp32 square root with a 1e-6 margin covers its own and the
// conversion's rounding and spares the FP64 pipe the ~10 instructions of a double-precision sqrt per particle-step.
__device__ __forceinline__ double step_len(double s2) { return (double)(sqrtf((float)s2) * 1.000001f); }
__device__ __forceinline__ float step_len(float s2) { return sqrtf(s2); }

// Branch-free pair term: the four pairs of a batch form four independent dependency chains.
template <typename T, bool ENERGY>
__device__ __forceinline__ void pair_term_nb(const Params<T>& p, bool valid, bool wall, T dx, T dy, T dz,
                                             Acc<T, ENERGY>& av, Acc<T, ENERGY>& aw)
{
    const T r2 = fma_(dz, dz, fma_(dy, dy, dx * dx));
    const bool hit = valid && r2 < p.rc2;                   // strict, same r^2 arithmetic as every other path
    const T inv = rcp_fast(hit ? r2 : T(1));
    T s3, s6, g;
    if (ENERGY) {
        const T s = (wall ? p.sig2_vw : p.sig2_vv) * inv;
        s3 = s * s * s;
        s6 = s3 * s3;
        g = hit ? (wall ? p.e24_vw : p.e24_vv) * inv * (T(2) * s6 - s3) : T(0);
    } else {                                                // time loop: 5 instead of 7 operations after 1 / r^2
        const T i3 = inv * inv * inv;
        g = hit ? fma_(wall ? p.c12_vw : p.c12_vv, i3, -(wall ? p.c6_vw : p.c6_vv)) * i3 * inv : T(0);
    }
    const T gw = wall ? g : T(0), gv = wall ? T(0) : g;
    if (ENERGY) {                                           // U_vv and U_vw are reported separately
        av.fx = fma_(gv, dx, av.fx); av.fy = fma_(gv, dy, av.fy); av.fz = fma_(gv, dz, av.fz);
        aw.fx = fma_(gw, dx, aw.fx); aw.fy = fma_(gw, dy, aw.fy); aw.fz = fma_(gw, dz, aw.fz);
    } else {                                                // time loop: one accumulator (aw stays 0)
        av.fx = fma_(g, dx, av.fx); av.fy = fma_(g, dy, av.fy); av.fz = fma_(g, dz, av.fz);
    }
    if (ENERGY) {
        const double u = hit ? (double)((wall ? p.e4_vw : p.e4_vv) * (s6 - s3) - (wall ? p.uc_vw : p.uc_vv)) : 0.0;
        const double w = (double)(g * r2);
        if (wall) { aw.u += u; aw.w += w; aw.c += hit; }
        else { av.u += u; av.w += w; av.c += hit; }
    }
}

// Batches of VL_BATCH list entries; while batch b is evaluated the indices of batch b + 1 are in flight.  The first
// index loads do not wait for the list length (rows beyond it are allocated; their values are masked), so the
// first positions are requested one round trip after the thread starts.
#ifndef MD_VL_BATCH
#define MD_VL_BATCH 4
#endif
constexpr int VL_BATCH = MD_VL_BATCH;
template <typename T, bool ENERGY, bool FOLD>
__device__ __forceinline__ void list_loop(const Params<T>& p, const int* __restrict__ lst, size_t stride, int n,
                                          const Vec4<T>* __restrict__ r, const Vec4<T>& ri, const int (&j0)[VL_BATCH],
                                          Acc<T, ENERGY>& av, Acc<T, ENERGY>& aw)
{
    const bool px = FOLD && p.bc[0] == BC_PERIODIC, py = FOLD && p.bc[1] == BC_PERIODIC, pz = FOLD && p.bc[2] == BC_PERIODIC;
    int jn[VL_BATCH];
#pragma unroll
    for (int u = 0; u < VL_BATCH; ++u) jn[u] = u < n ? j0[u] : -1;
    for (int k = 0; k < n; k += VL_BATCH) {
        int j[VL_BATCH];
        Vec4<T> rj[VL_BATCH];
#pragma unroll
        for (int u = 0; u < VL_BATCH; ++u) { j[u] = jn[u]; rj[u] = r[max(j[u], 0)]; }
#pragma unroll
        for (int u = 0; u < VL_BATCH; ++u)
            jn[u] = k + VL_BATCH + u < n ? lst[(size_t)(k + VL_BATCH + u) * stride] : -1;   // next batch
#pragma unroll
        for (int u = 0; u < VL_BATCH; ++u) {
            const T dx = px ? fold(ri.x, rj[u].x, p.L[0], T(0.5) * p.L[0]) : ri.x - rj[u].x;
            const T dy = py ? fold(ri.y, rj[u].y, p.L[1], T(0.5) * p.L[1]) : ri.y - rj[u].y;
            const T dz = pz ? fold(ri.z, rj[u].z, p.L[2], T(0.5) * p.L[2]) : ri.z - rj[u].z;
            pair_term_nb<T, ENERGY>(p, j[u] >= 0, j[u] >= p.nv, dx, dy, dz, av, aw);
        }
    }
}

template <typename T, bool ENERGY>
__device__ __forceinline__ void list_force(const Params<T>& p, const Verlet<T>& v, const Vec4<T>* __restrict__ r, int i,
                                           const Vec4<T>& ri, int raw, const int (&j0)[VL_BATCH],
                                           Acc<T, ENERGY>& av, Acc<T, ENERGY>& aw)
{
    const int* __restrict__ lst = v.nbr + i;
    // one loop per warp: if any lane's particle sits in a face cell every lane folds (the comparisons never fire
    // for the others); a per-lane choice would run the two loops one after the other in most warps, because a
    // warp's 32 cell-ordered particles span most of an x row and so nearly always include a face cell
    const bool fold = __any_sync(__activemask(), (raw & VL_FOLD) != 0) || (raw & VL_FOLD);
    if (fold) list_loop<T, ENERGY, true>(p, lst, v.stride, raw & VL_NMASK, r, ri, j0, av, aw);
    else list_loop<T, ENERGY, false>(p, lst, v.stride, raw & VL_NMASK, r, ri, j0, av, aw);
}

template <typename T, bool ENERGY>
__device__ __forceinline__ void list_force(const Params<T>& p, const Verlet<T>& v, const Vec4<T>* __restrict__ r, int i,
                                           const Vec4<T>& ri, Acc<T, ENERGY>& av, Acc<T, ENERGY>& aw)
{
    int j0[VL_BATCH];
#pragma unroll
    for (int u = 0; u < VL_BATCH; ++u) j0[u] = v.nbr[(size_t)u * v.stride + i];   // in flight together with ncnt (and r_i, v_i)
    list_force<T, ENERGY>(p, v, r, i, ri, v.ncnt[i], j0, av, aw);
}

// A heavy particle's list shared by the VL_GROUP lanes of a group: lane `sub` takes entries sub, sub + 8, sub + 16,
// ... of every 4 * VL_GROUP (one batch of four covers lists of up to that many entries); the caller sums the lanes' partial forces.
template <typename T, bool FOLD>
__device__ __forceinline__ void list_loop_group(const Params<T>& p, const int* __restrict__ lst, size_t stride, int n,
                                                int sub, const Vec4<T>* __restrict__ r, const Vec4<T>& ri,
                                                const int (&j0)[4], Acc<T, false>& av, Acc<T, false>& aw)
{
    const bool px = FOLD && p.bc[0] == BC_PERIODIC, py = FOLD && p.bc[1] == BC_PERIODIC, pz = FOLD && p.bc[2] == BC_PERIODIC;
    int jn[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) jn[u] = sub + VL_GROUP * u < n ? j0[u] : -1;
    for (int k = 0; k < n; k += 4 * VL_GROUP) {
        int j[4];
        Vec4<T> rj[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { j[u] = jn[u]; rj[u] = r[max(j[u], 0)]; }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int kk = k + 4 * VL_GROUP + sub + VL_GROUP * u;
            jn[u] = kk < n ? lst[(size_t)kk * stride] : -1;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const T dx = px ? fold(ri.x, rj[u].x, p.L[0], T(0.5) * p.L[0]) : ri.x - rj[u].x;
            const T dy = py ? fold(ri.y, rj[u].y, p.L[1], T(0.5) * p.L[1]) : ri.y - rj[u].y;
            const T dz = pz ? fold(ri.z, rj[u].z, p.L[2], T(0.5) * p.L[2]) : ri.z - rj[u].z;
            pair_term_nb<T, false>(p, j[u] >= 0, j[u] >= p.nv, dx, dy, dz, av, aw);
        }
    }
}

// What a thread keeps in registers across the grid barrier while it owns the same particle from step to step (the
// particles fit one wave, no rebuild in between): the position and velocity it has just written and the static head
// of the list, so that the next phase starts with the neighbours' position loads instead of a round trip of its own;
// likewise the particle, list head and (lane 0) velocity of the lane group's first heavy particle.
template <typename T>
struct Carry {
    Vec4<T> r;
    T vx, vy, vz;
    int raw, j0[VL_BATCH];
    bool valid = false;
    int nh, hi, hraw, hj[4];
    T hvx, hvy, hvz;
    bool nhvalid = false, hvalid = false;
};

// ---- phase: [forces] -> [kick completing the step] -> [kick + drift of the next step] -----------
// force: compute f from the list (else use the stored f(t));  kick: complete the current step (F3);
// drift: start the next step (F2).
template <typename T>
__device__ __forceinline__ void phase_step(const Params<T>& p, const Verlet<T>& v, int c, int cv, bool force,
                                           bool kick, bool drift, int req, int gtid, int gthreads,
                                           T lam, double* ksum, Carry<T>& cy, const bool cyon)
{
    const Vec4<T>* __restrict__ rcur = v.st[c].r;
    Vec4<T>* __restrict__ rnew = v.st[c ^ 1].r;
    const State<T>& s = v.st[cv];
    double kacc = 0.0;
    // F3 / F2 of particle i once its force is known (v already carries F4's factor); v and rn return what was stored
    auto integrate = [&](int i, const Vec4<T>& ri, T& vx, T& vy, T& vz, T fx, T fy, T fz, Vec4<T>& rn) {
        if (kick) {                                    // F3: v(t) = v(t - dt/2) + (dt/2m) f(t)
            vx = vx + p.hk * fx; vy = vy + p.hk * fy; vz = vz + p.hk * fz;
        }
        if (ksum) kacc += 0.5 * p.mass * ((double)vx * vx + (double)vy * vy + (double)vz * vz);
        if (drift) {                                   // F2: v(t + dt/2), r(t + dt)
            vx = vx + p.hk * fx; vy = vy + p.hk * fy; vz = vz + p.hk * fz;
            const T sx = p.dt * vx, sy = p.dt * vy, sz = p.dt * vz;
            rn.x = ri.x + sx; rn.y = ri.y + sy; rn.z = ri.z + sz;
            if (p.prism) {
                const T ro[3] = {ri.x, ri.y, ri.z};
                T rr[3] = {rn.x, rn.y, rn.z}, vh[3] = {vx, vy, vz};
                prism_reflect(p, ro, rr, vh);
                rn.x = rr[0]; rn.y = rr[1]; rn.z = rr[2]; vx = vh[0]; vy = vh[1]; vz = vh[2];
            }
            // periodic dimensions are left unwrapped until the next rebuild; reflection is immediate
            int* err = v.flags + VF_ESCAPE;
            if (p.bc[0] == BC_REFLECT) boundary(rn.x, vx, p.L[0], BC_REFLECT, err);
            if (p.bc[1] == BC_REFLECT) boundary(rn.y, vy, p.L[1], BC_REFLECT, err);
            if (p.bc[2] == BC_REFLECT) boundary(rn.z, vz, p.L[2], BC_REFLECT, err);
            rn.w = ri.w + step_len(sx * sx + sy * sy + sz * sz); // path length >= displacement
            if (rn.w > v.half_skin) v.flags[VF_REQ0 + req] = 1;
            rnew[i] = rn;
        }
        if (kick || drift || lam != T(1)) { s.vx[i] = vx; s.vy[i] = vy; s.vz[i] = vz; }
    };
    for (int i = gtid; i < p.nv; i += gthreads) {
        const bool kept = cyon && cy.valid;               // cyon only when this loop runs at most once
        Vec4<T> ri;
        T vx, vy, vz;
        int raw = 0, j0[VL_BATCH];
        if (kept) {
            ri = cy.r; vx = cy.vx; vy = cy.vy; vz = cy.vz; raw = cy.raw;
#pragma unroll
            for (int u = 0; u < VL_BATCH; ++u) j0[u] = cy.j0[u];
        } else {
            ri = rcur[i];
            vx = s.vx[i]; vy = s.vy[i]; vz = s.vz[i];    // issued early, consumed after the force loop
#pragma unroll
            for (int u = 0; u < VL_BATCH; ++u) j0[u] = force ? v.nbr[(size_t)u * v.stride + i] : 0;   // in flight together
            if (force) raw = v.ncnt[i];
        }
        vx = lam * vx; vy = lam * vy; vz = lam * vz;     // F4 of the step just completed (lam = 1 without thermostat)
        T fx, fy, fz;
        if (force) {
            if (raw & VL_HEAVY) {                        // the whole particle belongs to a lane group below
                if (cyon) { cy.raw = raw; cy.valid = drift; }
                continue;
            }
            Acc<T, false> av, aw;
            list_force<T, false>(p, v, rcur, i, ri, raw, j0, av, aw);
            fx = av.fx + aw.fx; fy = av.fy + aw.fy; fz = av.fz + aw.fz;
            if (!drift) { v.f.fx[i] = fx; v.f.fy[i] = fy; v.f.fz[i] = fz; }   // f is read back only after a phase without drift
        } else {
            fx = v.f.fx[i]; fy = v.f.fy[i]; fz = v.f.fz[i];
        }
        Vec4<T> rn = ri;
        integrate(i, ri, vx, vy, vz, fx, fy, fz, rn);
        if (cyon && force) {
            cy.r = rn; cy.vx = vx; cy.vy = vy; cy.vz = vz; cy.raw = raw;
#pragma unroll
            for (int u = 0; u < VL_BATCH; ++u) cy.j0[u] = j0[u];
            cy.valid = drift;
        }
    }
    if (force) {
        // Heavy particles (list longer than heavy_t: next to a wall, inside a cluster): one per group of VL_GROUP
        // lanes, so that no warp walks a list several times the typical length while the grid waits at the
        // barrier.  Group slots are numbered so that the blocks past the last particle (idle when the particles
        // fill less than one wave) take this work first and the rest is dealt round-robin over the other blocks,
        // one group per block and warp at a time.
        int nh;
        if (cyon && cy.nhvalid) nh = cy.nh;
        else {
            nh = min(v.flags[VF_NHEAVY], v.flags[VF_HCAP]);
            if (cyon) { cy.nh = nh; cy.nhvalid = true; }
        }
        const int lane = threadIdx.x & 31, sub = lane & (VL_GROUP - 1);
        const unsigned gmask = ((1u << VL_GROUP) - 1u) << (lane & ~(VL_GROUP - 1));
        constexpr int GPW = 32 / VL_GROUP, GPB = VL_THREADS / VL_GROUP;         // groups per warp, per block
        const int nbl = min((int)gridDim.x, (p.nv + VL_THREADS - 1) / VL_THREADS), nsp = (int)gridDim.x - nbl;
        const int b = blockIdx.x, q = (lane / VL_GROUP) * (VL_THREADS / 32) + (threadIdx.x >> 5);
        const int slot = b >= nbl ? (b - nbl) + nsp * ((threadIdx.x >> 5) * GPW + lane / VL_GROUP) : nsp * GPB + q * nbl + b;
        for (int h = slot; h < nh; h += gthreads / VL_GROUP) {
            const bool first = h == slot, kept = cyon && first && cy.hvalid;
            int i, raw, j0[4];
            T vx = T(0), vy = T(0), vz = T(0);
            if (kept) {
                i = cy.hi; raw = cy.hraw; vx = cy.hvx; vy = cy.hvy; vz = cy.hvz;
#pragma unroll
                for (int u = 0; u < 4; ++u) j0[u] = cy.hj[u];
            } else {
                i = v.cell[h]; raw = v.slot[h];
#pragma unroll
                for (int u = 0; u < 4; ++u) j0[u] = v.nbr[(size_t)(sub + VL_GROUP * u) * v.stride + i];
                if (sub == 0) { vx = s.vx[i]; vy = s.vy[i]; vz = s.vz[i]; }
            }
            const Vec4<T> ri = rcur[i];
            vx = lam * vx; vy = lam * vy; vz = lam * vz;
            Acc<T, false> av, aw;
            const bool fold = __any_sync(__activemask(), (raw & VL_FOLD) != 0) || (raw & VL_FOLD);
            if (fold) list_loop_group<T, true>(p, v.nbr + i, v.stride, raw & VL_NMASK, sub, rcur, ri, j0, av, aw);
            else list_loop_group<T, false>(p, v.nbr + i, v.stride, raw & VL_NMASK, sub, rcur, ri, j0, av, aw);
            T fx = av.fx + aw.fx, fy = av.fy + aw.fy, fz = av.fz + aw.fz;
#pragma unroll
            for (int o = 1; o < VL_GROUP; o <<= 1) {
                fx += __shfl_xor_sync(gmask, fx, o);
                fy += __shfl_xor_sync(gmask, fy, o);
                fz += __shfl_xor_sync(gmask, fz, o);
            }
            if (sub == 0) {
                if (!drift) { v.f.fx[i] = fx; v.f.fy[i] = fy; v.f.fz[i] = fz; }
                Vec4<T> rn = ri;
                integrate(i, ri, vx, vy, vz, fx, fy, fz, rn);
            }
            if (cyon && first) {
                cy.hi = i; cy.hraw = raw; cy.hvx = vx; cy.hvy = vy; cy.hvz = vz;
#pragma unroll
                for (int u = 0; u < 4; ++u) cy.hj[u] = j0[u];
                cy.hvalid = drift;
            }
        }
    }
    if (ksum) {                                        // thermostat: this thread's share of K(t), one atomic per warp
        kacc = warp_sum_d(kacc);
        if ((threadIdx.x & 31) == 0 && kacc != 0.0) atomicAdd(ksum, kacc);
    }
}

template <typename T>
__device__ __forceinline__ void phase_step(const Params<T>& p, const Verlet<T>& v, int c, int cv, bool force,
                                           bool kick, bool drift, int req, int gtid, int gthreads,
                                           T lam = T(1), double* ksum = nullptr)
{
    Carry<T> none;
    phase_step<T>(p, v, c, cv, force, kick, drift, req, gtid, gthreads, lam, ksum, none, false);
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
        if (tile_sum) {
            for (int k = threadIdx.x; k < t; k += SCAN_THREADS) off += tile_sum[k];
        } else {            // few tiles: sum the earlier counts directly and save a phase + barrier
            const int4* __restrict__ c4 = reinterpret_cast<const int4*>(count);     // t * SCAN_TILE is a multiple of 4
#pragma unroll 8
            for (int k = threadIdx.x; k < t * (SCAN_TILE / 4); k += SCAN_THREADS) {
                const int4 q = c4[k];
                off += q.x + q.y + q.z + q.w;
            }
        }
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
            if (base + k < n) start[base + k] = run;     // counts are cleared in the list-build phase
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
// vapor (j < nv) or wall (j = nv + k).  ROWS = 3^(d-1) lanes cooperate on one particle: lane `row` walks the
// cell row (cy+ky, cz+kz) -- its three cells are one contiguous range of the cell-ordered arrays -- and
// appends its hits through a shared-memory counter.  Positions are wrapped here, so distances fold.
template <typename T>
__device__ __forceinline__ void list_range(const Params<T>& p, const Vec4<T>* __restrict__ r, int jb, int je, int skip,
                                           const Vec4<T>& ri, T rl2, int* __restrict__ lst, size_t stride, int* cnt)
{
    const bool px = p.bc[0] == BC_PERIODIC, py = p.bc[1] == BC_PERIODIC, pz = p.bc[2] == BC_PERIODIC;
    constexpr int NB = 8;                                                // a cell row rarely holds more
    for (int j0 = jb; j0 < je; j0 += NB) {
        Vec4<T> rj[NB];
#pragma unroll
        for (int u = 0; u < NB; ++u) rj[u] = r[min(j0 + u, je - 1)];     // NB loads in flight
#pragma unroll
        for (int u = 0; u < NB; ++u) {
            const int j = j0 + u;
            const T dx = px ? fold(ri.x, rj[u].x, p.L[0], T(0.5) * p.L[0]) : ri.x - rj[u].x;
            const T dy = py ? fold(ri.y, rj[u].y, p.L[1], T(0.5) * p.L[1]) : ri.y - rj[u].y;
            const T dz = pz ? fold(ri.z, rj[u].z, p.L[2], T(0.5) * p.L[2]) : ri.z - rj[u].z;
            const T r2 = fma_(dz, dz, fma_(dy, dy, dx * dx));
            if (j < je && j != skip && r2 < rl2) {
                const int k = atomicAdd(cnt, 1);
                if (k < VL_MAXN) lst[(size_t)k * stride] = j;
            }
        }
    }
}

template <typename T, int ROWS>
__device__ __forceinline__ void phase_build(const Params<T>& p, const Verlet<T>& v, int c, int gtid, int gthreads, int hcap)
{
    constexpr int PPW = 32 / ROWS;                       // particles per warp
    __shared__ int s_cnt[(VL_THREADS / 32) * PPW];
    const Vec4<T>* __restrict__ r = v.st[c].r;
    const int nx = p.nc[0], ny = p.nc[1], nz = p.nc[2];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int pl = lane / ROWS, row = lane - pl * ROWS;
    const int warp = gtid >> 5, nwarps = gthreads >> 5;
    int* cnt = s_cnt + wib * PPW + min(pl, PPW - 1);
    for (int base = warp * PPW; base < p.nv; base += nwarps * PPW) {
        const int i = base + pl;
        const bool active = pl < PPW && i < p.nv;
        if (active && row == 0) *cnt = 0;
        __syncwarp();
        if (active) {
            const Vec4<T> ri = r[i];
            int cx, cy, cz;
            const int ci = cell_index(p, ri.x, ri.y, ri.z, cx, cy, cz);
            int* __restrict__ lst = v.nbr + i;
            int qy = cy + row % 3 - 1, qz = cz + (ROWS == 9 ? row / 3 - 1 : 0);
            bool ok = true;
            if (qz < 0) { ok = p.bc[2] == BC_PERIODIC; qz += nz; }
            else if (qz >= nz) { ok = p.bc[2] == BC_PERIODIC; qz -= nz; }
            if (qy < 0) { ok = ok && p.bc[1] == BC_PERIODIC; qy += ny; }
            else if (qy >= ny) { ok = ok && p.bc[1] == BC_PERIODIC; qy -= ny; }
            if (ok) {
                const int x0 = max(cx - 1, 0), x1 = min(cx + 1, nx - 1);
                int xw = -1;
                if (p.bc[0] == BC_PERIODIC) { if (cx == 0) xw = nx - 1; else if (cx == nx - 1) xw = 0; }
                const int rowc = (qz * ny + qy) * nx;
                const bool do_wall = p.nw > 0 && v.wnear[ci];
                const int jb = v.start[rowc + x0], je = v.start[rowc + x1 + 1];
                int jb2 = 0, je2 = 0, wb = 0, we = 0, wb2 = 0, we2 = 0;
                if (xw >= 0) { jb2 = v.start[rowc + xw]; je2 = v.start[rowc + xw + 1]; }
                if (do_wall) {
                    wb = v.wstart[rowc + x0]; we = v.wstart[rowc + x1 + 1];
                    if (xw >= 0) { wb2 = v.wstart[rowc + xw]; we2 = v.wstart[rowc + xw + 1]; }
                }
                list_range<T>(p, r, jb, je, i, ri, v.rl2, lst, v.stride, cnt);
                list_range<T>(p, r, jb2, je2, i, ri, v.rl2, lst, v.stride, cnt);
                list_range<T>(p, r, p.nv + wb, p.nv + we, -1, ri, v.rl2, lst, v.stride, cnt);
                list_range<T>(p, r, p.nv + wb2, p.nv + we2, -1, ri, v.rl2, lst, v.stride, cnt);
            }
        }
        __syncwarp();
        if (active && row == 0) {
            const int n = *cnt;
            const Vec4<T> ri = r[i];
            int cx, cy, cz;
            cell_index(p, ri.x, ri.y, ri.z, cx, cy, cz);
            const bool face = (p.bc[0] == BC_PERIODIC && (cx == 0 || cx == nx - 1)) ||
                              (p.bc[1] == BC_PERIODIC && (cy == 0 || cy == ny - 1)) ||
                              (p.bc[2] == BC_PERIODIC && (cz == 0 || cz == nz - 1));
            // a long list goes to a lane group while the idle blocks have groups left (the counter keeps the
            // demand; the host sizes the next launch by it); `cell` and `slot` are free until the next rebuild
            int raw = min(n, VL_MAXN) | (face ? VL_FOLD : 0);
            if (n > v.heavy_t) {
                const int h = atomicAdd(v.flags + VF_NHEAVY, 1);
                if (h < hcap) { raw |= VL_HEAVY; v.cell[h] = i; v.slot[h] = raw; }
            }
            v.ncnt[i] = raw;
            if (n > VL_MAXN) v.flags[VF_OVERFLOW] = 1;
        }
        __syncwarp();
    }
}

// ---- the persistent time loop ---------------------------------------------------------------------
// md_step(n): phase(stored f; kick + drift), then n - 1 fused phases (force; kick; kick + drift), then
// phase(force; kick): n + 1 phases and n grid barriers for n steps, plus 5 barriers per rebuild.
// force_rebuild (md_create): bin + build the list first, then evaluate f(0).
// MINB = resident blocks per SM the register budget is sized for: 2 (up to 128 registers, the latency-bound
// sizes that fit one wave) or 3 (more warps to hide HBM latency once the state no longer fits in L2).
template <typename T, int ROWS, int MINB>
__global__ void __launch_bounds__(VL_THREADS, MINB) k_md_run(Params<T> p, Verlet<T> v, long long n_steps, int force_rebuild)
{
    unsigned long long bar_target = 0;
    const bool thermo = p.thermo_rate > 0.0;
    const int gtid = blockIdx.x * blockDim.x + threadIdx.x;
    const int gthreads = gridDim.x * blockDim.x;
    int c = v.flags[VF_CUR], cv = v.flags[VF_CURV];
    bool rebuild = force_rebuild != 0;
    Carry<T> carry;
    const bool cyon = MINB == 2 && v.carry && !thermo && gthreads >= p.nv;      // (the 3-blocks-per-SM variant serves N > one wave)
    // lane groups in the blocks past the last particle (none once the particles fill the grid)
    const int hcap = max((int)gridDim.x - (p.nv + VL_THREADS - 1) / VL_THREADS, 0) * (VL_THREADS / VL_GROUP);
    unsigned long long t0 = gtid == 0 ? now_ns() : 0ull, t1;
    for (long long s = 0;; ++s) {
        if (rebuild) {
            unsigned long long u0 = gtid == 0 ? now_ns() : 0ull, u1;
            if (gtid == 0) { v.flags[VF_NHEAVY] = 0; v.flags[VF_HCAP] = hcap; }
            phase_bin<T>(p, v, c, gtid, gthreads);
            grid_barrier(v.bar, bar_target);
            if (gtid == 0) { u1 = now_ns(); v.times[4] += u1 - u0; u0 = u1; }
            const bool two_level = p.ncell > 64 * SCAN_TILE;
            if (two_level) {
                phase_scan_reduce(v.count, p.ncell, v.tile_sum);
                grid_barrier(v.bar, bar_target);
            }
            phase_scan_apply(v.count, p.ncell, two_level ? v.tile_sum : nullptr, v.start);
            grid_barrier(v.bar, bar_target);
            if (gtid == 0) { u1 = now_ns(); v.times[5] += u1 - u0; u0 = u1; }
            phase_scatter<T>(p, v, c, cv, gtid, gthreads);
            grid_barrier(v.bar, bar_target);
            if (gtid == 0) { u1 = now_ns(); v.times[6] += u1 - u0; u0 = u1; }
            c ^= 1; cv ^= 1;
            phase_build<T, ROWS>(p, v, c, gtid, gthreads, hcap);
            for (int q = gtid; q < p.ncell; q += gthreads) v.count[q] = 0;                  // for the next rebuild
            if (gtid == 0) v.flags[VF_NREBUILD] += 1;
            grid_barrier(v.bar, bar_target);
            if (gtid == 0) { t1 = now_ns(); v.times[2] += t1 - t0; t0 = t1; v.times[7] += t1 - u0; }
            carry.valid = carry.hvalid = carry.nhvalid = false;          // new particle order, new lists
        }
        if (s == n_steps) break;
        const int req = (int)(s % 3);
        if (gtid == 0) { v.flags[VF_REQ0 + (req + 1) % 3] = 0; if (thermo) v.ksum[(s + 1) % 3] = 0.0; }   // slots of step s + 1
        unsigned long long dbg0 = 0;
        if (v.dbg) dbg0 = now_ns();
        if (!thermo || s == 0) {
            phase_step<T>(p, v, c, cv, s > 0, s > 0, true, req, gtid, gthreads, T(1), nullptr, carry, cyon);
        } else {
            // with the thermostat lambda(t) needs K(t) of ALL particles before the next drift: the fused phase splits
            // into [F1 + F3 + K partial sums] | barrier | [F4 rescale + F2], one extra barrier per step
            phase_step<T>(p, v, c, cv, true, true, false, req, gtid, gthreads, T(1), v.ksum + s % 3);
            grid_barrier(v.bar, bar_target);
            const double lam = berendsen_lambda(*(volatile double*)(v.ksum + s % 3), p.thermo_rate, p.t_target, p.dof);
            phase_step<T>(p, v, c, cv, false, false, true, req, gtid, gthreads, (T)lam);
        }
        if (v.dbg && (threadIdx.x & 31) == 0) atomicAdd(v.dbg + (gtid >> 5), now_ns() - dbg0);
        if (gtid == 0) { t1 = now_ns(); v.times[0] += t1 - t0; t0 = t1; }
        grid_barrier(v.bar, bar_target);
        if (gtid == 0) { t1 = now_ns(); v.times[1] += t1 - t0; t0 = t1; }
        c ^= 1;
        rebuild = *(volatile int*)(v.flags + VF_REQ0 + req) != 0;
    }
    if (thermo && n_steps > 0) {
        double* ks = v.ksum + n_steps % 3;
        phase_step<T>(p, v, c, cv, true, true, false, 0, gtid, gthreads, T(1), ks);
        grid_barrier(v.bar, bar_target);
        const double lam = berendsen_lambda(*(volatile double*)ks, p.thermo_rate, p.t_target, p.dof);
        phase_step<T>(p, v, c, cv, false, false, false, 0, gtid, gthreads, (T)lam);      // F4 of the last step
    } else if (n_steps > 0 || force_rebuild) {
        phase_step<T>(p, v, c, cv, true, n_steps > 0, false, 0, gtid, gthreads);
    }
    if (gtid == 0) { v.flags[VF_CUR] = c; v.flags[VF_CURV] = cv; v.times[3] += now_ns() - t0; }
}

// Diagnostics only (MD_DEBUG_BUILD=1 in md_profile_step): the list-build phase as a kernel of its own, so that ncu can
// attribute its stalls.  It rebuilds the list from the current cell order, which is what the list already holds.
template <typename T, int ROWS>
__global__ void __launch_bounds__(VL_THREADS, 2) k_dbg_build(Params<T> p, Verlet<T> v, int c)
{
    phase_build<T, ROWS>(p, v, c, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x, v.flags[VF_HCAP]);
}

// Diagnostics only (MD_DEBUG_BUILD=1): the force part of the step phase as a kernel of its own (recomputes f(t)).
template <typename T>
__global__ void __launch_bounds__(VL_THREADS, 2) k_dbg_force(Params<T> p, Verlet<T> v, int c, int cv)
{
    phase_step<T>(p, v, c, cv, true, false, false, 0, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
}

// a5 energy pass over the neighbour list (ordinary launch; the host passes the buffer parities).
template <typename T>
__global__ void __launch_bounds__(VL_THREADS) k_verlet_energy(Params<T> p, Verlet<T> v, int c, EnergyOut eo)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.nv) return;
    const Vec4<T>* __restrict__ r = v.st[c].r;
    const Vec4<T> ri = r[i];
    Acc<T, true> av, aw;
    list_force<T, true>(p, v, r, i, ri, av, aw);
    eo.pe[i] = 0.5 * av.u + aw.u;
    eo.pew[i] = aw.u;
    eo.vir[i] = 0.5 * av.w + aw.w;
    eo.cvv[i] = av.c;
    eo.cvw[i] = aw.c;
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
