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
//
// Round 2 (profiles/r02_*.md): (i) the list build runs its distance filter in FP32 on a float4 shadow of the positions
// (the list only has to be a SUPERSET of the pairs within r_c + skin; the force loop still takes the r < r_c decision in
// full precision); (ii) periodic images are materialised as ghost copies the owner rewrites in its drift, so the time loop
// never folds a difference; (iii) a list holds its vapor entries from the first slot up and its wall entries from the last
// slot down, so the pair loop carries one set of coefficients at a time; (iv) lists are stored warp-blocked with a constant
// stride between a particle's entries; (v) the grid barrier is a release reduction plus one acquire load and carries the
// rebuild request; (vi) TWO-LEVEL LIST: between two full rebuilds (bin, scan, scatter, cell walk) the r_c + skin list is
// pruned from an outer list of the pairs within r_c + outer skin (phase_prune), exactly.
#pragma once
#include "md_kernels.cuh"

namespace md {

#ifndef MD_VL_THREADS
#define MD_VL_THREADS 256
#endif
constexpr int VL_THREADS = MD_VL_THREADS;   // threads per block of the persistent kernel
constexpr int VS_ITEMS = 8, VS_TILE = VL_THREADS * VS_ITEMS;   // in-kernel scan: counts per thread, per tile
constexpr int VL_MAXN = 128;   // neighbour-list entries per particle
constexpr int VL_MAXO = 256;   // outer-list entries per particle (two-level list, see phase_prune)
// List layout: warp-blocked.  The lists of particles 32 b .. 32 b + 31 form one block of MAXK rows of 32 entries: entry k of
// particle i sits at ((i / 32) MAXK + k) 32 + i % 32.  A warp's loads of entry k are one 128-byte line, as in the fully
// transposed layout of round 1 (k stride = N_v), but consecutive entries of a particle are a CONSTANT 128 bytes apart, so
// a list walk is immediate offsets from one base pointer instead of a 64-bit multiply-add per entry: a third of the
// instructions of the prune and a tenth of the step loop were that address arithmetic (profiles/r02_k_md_run.md).
constexpr int VL_LS = 32;
__device__ __forceinline__ size_t vl_base(int i, int maxk) { return ((size_t)(i >> 5) * maxk << 5) + (i & 31); }

// flags: (slots 0-2 unused: the rebuild request now travels in the grid barrier's word), list overflow, position-buffer parity, velocity/id-buffer parity, rebuild count, escape,
// particles with a long list at the last rebuild (demand), how many of them the idle blocks' lane groups took (capacity),
// the same two for the lists long enough for a whole warp
// The two heavy-list counters exist twice (+ parity of the list event that filled them: a prune fills the set the step
// phases are not reading, and the set just retired is cleared one barrier before anybody can write it again); VF_HPAR =
// the parity in use when the launch ended; VF_OUTER_BAD = the last outer list overflowed (no pruning until the next
// outer build); VF_NOHEAVY = particles with a long OUTER list (pruned by a warp each); VF_NPRUNE = prunes so far.
enum { VF_UNUSED0 = 0, VF_OVERFLOW = 3, VF_CUR = 4, VF_CURV = 5, VF_NREBUILD = 6, VF_ESCAPE = 7, VF_NHEAVY = 8, VF_HCAP = 10,
       VF_NHEAVY32 = 11, VF_HCAP32 = 13, VF_HPAR = 14, VF_OUTER_BAD = 15, VF_NOHEAVY = 16, VF_NPRUNE = 17 /* + 1: prunes since the last full rebuild */, VF_COUNT = 19 };

// Shadow entry of the list build: (x, y, z) rounded to fp32.
struct alignas(16) F4 {
    float x, y, z, w;
};

template <typename T>
struct Verlet {
    // st[c].r: positions, double-buffered every step.  Layout of one buffer: nimg image blocks of ntot = nv + nw
    // entries each; block 0 holds the particles themselves (nv vapor entries in cell order, then the nw wall
    // entries in cell order, static), block m > 0 the copies shifted by -+L in the dimensions whose bit is set in
    // m (written only for particles in the first / last cell of those dimensions: the ghosts).
    // st[cv].{vx,vy,vz,id}: owner-only data, swapped only by the rebuild's scatter
    State<T> st[2];
    Force<T> f;
    int *nbr, *ncnt;           // nbr[vl_base(i, VL_MAXN) + k * VL_LS], k < VL_MAXN: index into a position buffer; ncnt[nv]: see VL_* below
    // two-level list (nprune > 0): onbr[vl_base(i, VL_MAXO) + k * VL_LS], k < VL_MAXO = every j within r_c + outer skin of i at the last
    // full rebuild; ocnt = its counts (VO_*); oheavy = particles whose outer list a whole warp prunes; wo = path of i
    // between the last full rebuild and the last list event (owner-only)
    int *onbr, *ocnt, *oheavy;
    T* wo;
    int *cell, *slot, *count, *start;
    unsigned long long* tile_agg;   // scan: (rebuild generation, sum of the tile's counts) per tile of VS_TILE cells
    const int* wstart;         // walls: [ncell + 1] ranges into the wall part of an image block
    const uint8_t* wnear;
    F4* r32;                   // [ntot] fp32 shadow of image block 0 (vapor part rewritten by every scatter); T = double only
    int* flags;                // VF_*
    unsigned long long* bar;   // grid barrier arrival counter
    double* ksum;              // [3] kinetic-energy accumulators of the thermostat, rotating over the steps (a slot is
                               // cleared one barrier before the phase that adds to it and read one barrier after)
    unsigned long long* dbg;   // optional per-warp step-phase ns (diagnostics build), or nullptr
    unsigned long long* times; // [10] ns seen by thread 0: step phases, step barriers, list events, final phase,
                               // full-rebuild split: bin, scan, scatter, list build (each with its barrier); [8] prunes
    T half_skin;               // skin / 2
    float rl2f;                // (r_c + skin)^2 plus the fp32 rounding of the filter (positions, image shift, fma chain)
    float rl2f_out;            // the same for r_c + outer skin
    T rl2_prune;               // (r_c + skin)^2 for the prune's test on the positions themselves
    T outer_lim;               // (outer skin - skin) / 2: a prune is valid while no path since the full rebuild exceeds it
    int nprune;                // prunes allowed between two full rebuilds (0: single-level list)
    int ntot, nimg;            // image-block stride nv + nw; number of image blocks (1 in fp32 mode: that mode folds)
    int carry;                 // 0: reload own state every step (diagnostic A/B)
    int heavy_t;               // particles whose list is longer than this are "heavy": in the step phase a group of
                               // VL_GROUP lanes shares one such list (indices in `cell`, ncnt words in `slot` -- both
                               // free between rebuilds; their number in flags[VF_NHEAVY]), a whole warp if it is
                               // longer than VL_WARP_T (registered from the top of `cell` / `slot` downwards)
};

// ncnt word of a particle: vapor entries in list slots [0, nvv), wall entries in the LAST nvw slots [VL_MAXN - nvw,
// VL_MAXN) (the two are appended by different warps of the build, from the two ends); face code = 2 bits
// per dimension, 1 = the particle sat in the FIRST cell of a periodic dimension when the list was built (its ghost is
// the copy at +L), 2 = in the LAST cell (ghost at -L); heavy = list walked by a lane group (see phase_step).
constexpr int VL_NVV_MASK = 0xff, VL_NVW_SHIFT = 8, VL_NVW_MASK = 0xff, VL_FACE_SHIFT = 16, VL_FACE_MASK = 0x3f;
constexpr int VL_HEAVY = 1 << 29;
// ocnt word: vapor entries in outer slots [0, ov), wall entries in the last ow slots, the face code, "pruned by a warp"
constexpr int VO_MASK = 0x3ff, VO_W_SHIFT = 10, VO_FACE_SHIFT = 20, VO_HEAVY = 1 << 30;
#ifndef MD_VO_HEAVY_T
#define MD_VO_HEAVY_T 40
#endif
constexpr int VO_HEAVY_T = MD_VO_HEAVY_T;          // outer lists longer than this (mean 17 at density 0.05) are pruned by a whole warp
__device__ __forceinline__ int vl_nvv(int raw) { return raw & VL_NVV_MASK; }
__device__ __forceinline__ int vl_nvw(int raw) { return (raw >> VL_NVW_SHIFT) & VL_NVW_MASK; }
__device__ __forceinline__ int vl_face(int raw) { return (raw >> VL_FACE_SHIFT) & VL_FACE_MASK; }
#ifndef MD_VL_GROUP
#define MD_VL_GROUP 4
#endif
constexpr int VL_GROUP = MD_VL_GROUP;   // lanes sharing one heavy particle's list
#ifndef MD_VL_WARP_T
#define MD_VL_WARP_T 48
#endif
constexpr int VL_WARP_T = MD_VL_WARP_T;   // lists longer than this (inside an adsorbed film: up to ~100 entries) get a whole warp
#ifndef MD_VL_WARP_ROUNDS
#define MD_VL_WARP_ROUNDS 1
#endif
constexpr int VL_WARP_ROUNDS = MD_VL_WARP_ROUNDS;       // such lists per idle warp and step

// d = a - b folded to the nearest image by comparison (|true d| < r_c + skin < L/2): fp32 mode only, where a ghost
// copy x + L would round the coordinate.  The shift goes on whichever particle sits at the top of the box so the
// difference stays exact.
__device__ __forceinline__ float fold(float a, float b, float L, float halfL)
{
    float d = a - b;
    if (d > halfL) d = (a - L) - b;
    else if (d < -halfL) d = a - (b - L);
    return d;
}
__device__ __forceinline__ double fold(double a, double b, double, double) { return a - b; }   // never used: fp64 reads ghosts

// Grid barrier of the cooperative launch (all blocks are co-resident), which also carries the step's one global
// decision.  One arrival per block: a release reduction (MEMBAR.ALL.GPU + REDG; __threadfence() + atomicAdd was a
// sequentially consistent fence, an L1 invalidation that also evicts the lines of the other block still computing on the
// SM, and an atomic with a return value), relaxed polling, and ONE acquire load when released (LDG + CCTL.IVALL) --
// cooperative_groups' grid.sync() re-acquires on every poll (profiles/r01_v3_cfg2.md).  A flag per block polled by every
// block (no atomic) was measured in round 2 and is 4x slower at 296 blocks (profiles/r02_k_md_run.md).
// The 64-bit word: arrivals in bits 0..39, and two 12-bit fields that count the blocks asking for a rebuild at even and
// at odd barriers.  A block reads the field of the barrier's own parity: the other blocks can only have added to it at
// this barrier (nobody reaches the barrier after the next before everybody has left this one), so every block takes the
// same decision -- what the three rotating request slots in global memory and a load after every barrier did before.
// `bar` is zeroed by the host before every launch.
struct GridBarrier {
    unsigned long long target = 0;     // arrivals expected when the current barrier completes (thread 0 only)
    unsigned int seen_req[2] = {0, 0}; // last value of the two request fields (thread 0 only)
    unsigned int index = 0;            // barriers passed so far
};

__device__ __forceinline__ bool grid_barrier(unsigned long long* bar, GridBarrier& g, bool request = false)
{
    __shared__ int s_any;
    const int par = g.index & 1;
    ++g.index;
    const int mine = __syncthreads_or(request);
    if (threadIdx.x == 0) {
        g.target += gridDim.x;
        const unsigned long long add = 1ull + (mine ? 1ull << (40 + 12 * par) : 0ull);
        asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(bar), "l"(add) : "memory");
        unsigned long long seen;
        do {
            asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(seen) : "l"(bar) : "memory");
        } while ((seen & ((1ull << 40) - 1ull)) < g.target);
        asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(seen) : "l"(bar) : "memory");   // later loads see every block's writes
        const unsigned int field = (unsigned int)(seen >> (40 + 12 * par)) & 0xfffu;
        s_any = field != g.seen_req[par];
        g.seen_req[par] = field;
    }
    __syncthreads();
    return s_any != 0;
}

__device__ __forceinline__ unsigned long long now_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}

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

// Coefficients of one pair type (vapor-vapor or vapor-wall), held in registers by the pair loop.
template <typename T>
struct PairCoef {
    T rc2, c12, c6;            // time loop: g = (c12 / r^6 - c6) / r^8
    T sig2, e24, e4, uc;       // energy pass: the oracle's s = sigma^2 / r^2 form
};
template <typename T>
__device__ __forceinline__ PairCoef<T> coef_vv(const Params<T>& p) { return {p.rc2, p.c12_vv, p.c6_vv, p.sig2_vv, p.e24_vv, p.e4_vv, p.uc_vv}; }
template <typename T>
__device__ __forceinline__ PairCoef<T> coef_vw(const Params<T>& p) { return {p.rc2, p.c12_vw, p.c6_vw, p.sig2_vw, p.e24_vw, p.e4_vw, p.uc_vw}; }

// Branch-free pair term: the pairs of a batch form independent dependency chains.
template <typename T, bool ENERGY>
__device__ __forceinline__ void pair_term_nb(const PairCoef<T>& q, bool valid, T dx, T dy, T dz, Acc<T, ENERGY>& a)
{
    const T r2 = fma_(dz, dz, fma_(dy, dy, dx * dx));
    const bool hit = valid && r2 < q.rc2;                   // strict, same r^2 arithmetic as every other path
    const T inv = rcp_fast(hit ? r2 : T(1));
    T s3, s6, g;
    if (ENERGY) {
        const T s = q.sig2 * inv;
        s3 = s * s * s;
        s6 = s3 * s3;
        g = hit ? q.e24 * inv * (T(2) * s6 - s3) : T(0);
    } else {                                                // time loop: 5 instead of 7 operations after 1 / r^2
        const T i3 = inv * inv * inv;
        g = hit ? fma_(q.c12, i3, -q.c6) * i3 * inv : T(0);
    }
    a.fx = fma_(g, dx, a.fx); a.fy = fma_(g, dy, a.fy); a.fz = fma_(g, dz, a.fz);
    if (ENERGY) {
        a.u += hit ? (double)(q.e4 * (s6 - s3) - q.uc) : 0.0;
        a.w += (double)(g * r2);
        a.c += hit;
    }
}

// One segment (vapor or wall) of a particle's list, one thread per particle.  The list is stored transposed,
// nbr[k * stride + i], so a warp's loads of entry k are coalesced.  Entries are consumed VL_BATCH at a time: that many
// index loads, then position loads, are in flight together, and while batch b is evaluated the indices of batch b + 1
// are in flight.  The first index loads do not wait for the list length (rows beyond it are allocated; their values
// are masked).  fp64: an entry already names the image (ghost copy) to read, differences are plain.  fp32: FOLD.
#ifndef MD_VL_BATCH
#define MD_VL_BATCH 4
#endif
constexpr int VL_BATCH = MD_VL_BATCH;
template <typename T, bool ENERGY, bool FOLD>
__device__ __forceinline__ void list_loop(const Params<T>& p, const PairCoef<T>& q, const int* __restrict__ lst,
                                          int n, const Vec4<T>* __restrict__ r, const Vec4<T>& ri, const int (&j0)[VL_BATCH],
                                          Acc<T, ENERGY>& a)
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
            jn[u] = k + VL_BATCH + u < n ? lst[(k + VL_BATCH + u) * VL_LS] : -1;   // next batch
#pragma unroll
        for (int u = 0; u < VL_BATCH; ++u) {
            const T dx = px ? fold(ri.x, rj[u].x, p.L[0], T(0.5) * p.L[0]) : ri.x - rj[u].x;
            const T dy = py ? fold(ri.y, rj[u].y, p.L[1], T(0.5) * p.L[1]) : ri.y - rj[u].y;
            const T dz = pz ? fold(ri.z, rj[u].z, p.L[2], T(0.5) * p.L[2]) : ri.z - rj[u].z;
            pair_term_nb<T, ENERGY>(q, j[u] >= 0, dx, dy, dz, a);
        }
    }
}

// Both segments of particle i's list: vapor entries (first VL_BATCH indices already in j0), then wall entries.  One
// loop variant per warp: in fp32 mode every lane folds if any lane's particle sat in a face cell when the list was
// built (a per-lane choice would run the two loops one after the other in most warps, because a warp's 32
// cell-ordered particles span most of an x row and so nearly always include a face cell).
template <typename T, bool ENERGY>
__device__ __forceinline__ void list_force(const Params<T>& p, const Verlet<T>& v, const Vec4<T>* __restrict__ r, int i,
                                           const Vec4<T>& ri, int raw, const int (&j0)[VL_BATCH],
                                           Acc<T, ENERGY>& av, Acc<T, ENERGY>& aw)
{
    const int* __restrict__ lst = v.nbr + vl_base(i, VL_MAXN);
    const int nvv = vl_nvv(raw), nvw = vl_nvw(raw);
    const bool fold = sizeof(T) == 4 && __any_sync(__activemask(), vl_face(raw) != 0);
    const PairCoef<T> qv = coef_vv(p);
    if (fold) list_loop<T, ENERGY, true>(p, qv, lst, nvv, r, ri, j0, av);
    else list_loop<T, ENERGY, false>(p, qv, lst, nvv, r, ri, j0, av);
    if (__any_sync(__activemask(), nvw != 0)) {             // walls: a few per cent of the particles have any
        const PairCoef<T> qw = coef_vw(p);
        const int* __restrict__ lw = lst + (VL_MAXN - nvw) * VL_LS;
        int w0[VL_BATCH];
#pragma unroll
        for (int u = 0; u < VL_BATCH; ++u) w0[u] = u < nvw ? lw[u * VL_LS] : -1;
        if (fold) list_loop<T, ENERGY, true>(p, qw, lw, nvw, r, ri, w0, aw);
        else list_loop<T, ENERGY, false>(p, qw, lw, nvw, r, ri, w0, aw);
    }
}

template <typename T, bool ENERGY>
__device__ __forceinline__ void list_force(const Params<T>& p, const Verlet<T>& v, const Vec4<T>* __restrict__ r, int i,
                                           const Vec4<T>& ri, Acc<T, ENERGY>& av, Acc<T, ENERGY>& aw)
{
    int j0[VL_BATCH];
#pragma unroll
    for (int u = 0; u < VL_BATCH; ++u) j0[u] = v.nbr[vl_base(i, VL_MAXN) + u * VL_LS];   // in flight together with ncnt (and r_i, v_i)
    list_force<T, ENERGY>(p, v, r, i, ri, v.ncnt[i], j0, av, aw);
}

// A heavy particle's list shared by the VL_GROUP lanes of a group: lane `sub` takes entries sub, sub + VL_GROUP, ... of
// every 4 * VL_GROUP (one batch of four covers lists of up to that many entries); the caller sums the lanes' partial
// forces.  Vapor and wall entries are told apart by their slot (k < nvv), so this loop selects the coefficients per
// entry -- the price of sharing one list, paid only by the few heavy particles.
template <typename T, bool FOLD>
__device__ __forceinline__ void list_loop_group(const Params<T>& p, const int* __restrict__ lst, int nvv, int n,
                                                int sub, const Vec4<T>* __restrict__ r, const Vec4<T>& ri,
                                                const int (&j0)[4], Acc<T, false>& a)
{
    const bool px = FOLD && p.bc[0] == BC_PERIODIC, py = FOLD && p.bc[1] == BC_PERIODIC, pz = FOLD && p.bc[2] == BC_PERIODIC;
    const PairCoef<T> qv = coef_vv(p), qw = coef_vw(p);
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
            jn[u] = kk < n ? lst[(kk < nvv ? kk : kk + VL_MAXN - n) * VL_LS] : -1;   // wall entries sit at the top
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const T dx = px ? fold(ri.x, rj[u].x, p.L[0], T(0.5) * p.L[0]) : ri.x - rj[u].x;
            const T dy = py ? fold(ri.y, rj[u].y, p.L[1], T(0.5) * p.L[1]) : ri.y - rj[u].y;
            const T dz = pz ? fold(ri.z, rj[u].z, p.L[2], T(0.5) * p.L[2]) : ri.z - rj[u].z;
            const bool wall = k + sub + VL_GROUP * u >= nvv;
            PairCoef<T> q;
            q.rc2 = qv.rc2; q.c12 = wall ? qw.c12 : qv.c12; q.c6 = wall ? qw.c6 : qv.c6;
            pair_term_nb<T, false>(q, j[u] >= 0, dx, dy, dz, a);
        }
    }
}

// Ghost copies of particle i (fp64): position `rn` shifted by +L (face code 1) or -L (face code 2) in every non-empty
// subset of the dimensions in which the particle sat in a face cell when the list was built; image block m (bit a =
// dimension a shifted) holds the copy.  Only these copies are ever read: a list entry names one when the build
// reached the neighbour across a periodic face.
template <typename T>
__device__ __forceinline__ void write_ghosts(const Params<T>& p, const Verlet<T>& v, Vec4<T>* __restrict__ r, int i,
                                             const Vec4<T>& rn, int face)
{
    const int dims = ((face & 3) ? 1 : 0) | ((face & 12) ? 2 : 0) | ((face & 48) ? 4 : 0);
    const T sx = (face & 3) == 1 ? p.L[0] : -p.L[0], sy = ((face >> 2) & 3) == 1 ? p.L[1] : -p.L[1],
            sz = ((face >> 4) & 3) == 1 ? p.L[2] : -p.L[2];
    for (int m = 1; m < v.nimg; ++m) {
        if (m & ~dims) continue;
        Vec4<T> g;
        g.x = (m & 1) ? rn.x + sx : rn.x;
        g.y = (m & 2) ? rn.y + sy : rn.y;
        g.z = (m & 4) ? rn.z + sz : rn.z;
        g.w = T(0);
        r[(size_t)m * v.ntot + i] = g;
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
    int nh, n32, hi, hraw, hj[4];
    T hvx, hvy, hvz;
    bool nhvalid = false, hvalid = false;
};

// ---- phase: [forces] -> [kick completing the step] -> [kick + drift of the next step] -----------
// force: compute f from the list (else use the stored f(t));  kick: complete the current step (F3);
// drift: start the next step (F2).
template <typename T>
__device__ __forceinline__ void phase_step(const Params<T>& p, const Verlet<T>& v, int c, int cv, bool force,
                                           bool kick, bool drift, bool& want, int gtid, int gthreads, int hp,
                                           T lam, double* ksum, Carry<T>& cy, const bool cyon)
{
    constexpr bool GHOSTS = sizeof(T) == 8;
    const Vec4<T>* __restrict__ rcur = v.st[c].r;
    Vec4<T>* __restrict__ rnew = v.st[c ^ 1].r;
    const State<T>& s = v.st[cv];
    double kacc = 0.0;
    // F3 / F2 of particle i once its force is known (v already carries F4's factor); v and rn return what was stored
    auto integrate = [&](int i, const Vec4<T>& ri, T& vx, T& vy, T& vz, T fx, T fy, T fz, Vec4<T>& rn, int face) {
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
            if (rn.w > v.half_skin) want = true;
            rnew[i] = rn;
            if (GHOSTS && face) write_ghosts(p, v, rnew, i, rn, face);
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
            for (int u = 0; u < VL_BATCH; ++u) j0[u] = force ? v.nbr[vl_base(i, VL_MAXN) + u * VL_LS] : 0;   // in flight together
            raw = v.ncnt[i];                             // the face code is needed by the drift even without a force pass
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
        integrate(i, ri, vx, vy, vz, fx, fy, fz, rn, vl_face(raw));
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
        int nh, n32;
        if (cyon && cy.nhvalid) { nh = cy.nh; n32 = cy.n32; }
        else {
            nh = min(v.flags[VF_NHEAVY + hp], v.flags[VF_HCAP]);
            n32 = min(v.flags[VF_NHEAVY32 + hp], v.flags[VF_HCAP32]);
            if (cyon) { cy.nh = nh; cy.n32 = n32; cy.nhvalid = true; }
        }
        const int lane = threadIdx.x & 31, sub = lane & (VL_GROUP - 1);
        const unsigned gmask = ((1u << VL_GROUP) - 1u) << (lane & ~(VL_GROUP - 1));
        constexpr int GPW = 32 / VL_GROUP, GPB = VL_THREADS / VL_GROUP;         // groups per warp, per block
        const int nbl = min((int)gridDim.x, (p.nv + VL_THREADS - 1) / VL_THREADS), nsp = (int)gridDim.x - nbl;
        const int b = blockIdx.x, q = (lane / VL_GROUP) * (VL_THREADS / 32) + (threadIdx.x >> 5);
        // Lists longer than VL_WARP_T (a particle inside an adsorbed film has ~100 neighbours within r_c + skin): one
        // per WARP, lane l takes entries l, l + 32, l + 64, l + 96 -- one batch, a butterfly sum, and lane 0 integrates.
        // Walked by four lanes such a list would take 7 batches while the grid waits.  The warps of the idle blocks that
        // hold no lane group take VL_WARP_ROUNDS each first (the group slots below fill every idle block's warps from
        // warp 0 up, these lists from its last warp down: a warp with eight groups AND such a list was the slowest of
        // the grid, 6.2 us against 4.8, once a film covers the wall); the rest goes to the warps of the particle blocks,
        // one each after their own particles (the film has ~1,500 such lists at N = 65,536, the idle blocks 320 warps).
        if (n32 > 0) {
            constexpr int WPB = VL_THREADS / 32;
            const int wi = threadIdx.x >> 5, back = WPB - 1 - wi;
            const int nfree = nsp > 0 ? max(WPB - (nh + nsp * GPW - 1) / (nsp * GPW), 0) : 0;   // idle warps per block without groups
            const int icap = nsp * nfree * VL_WARP_ROUNDS;
            const bool idle = b >= nbl;
            // idle blocks: block after block, last warp first; particle blocks likewise (spilled lane groups start at warp 0)
            const int h0 = idle ? (back < nfree ? (b - nbl) + nsp * back : n32) : icap + back * nbl + b;
            const int hlim = idle ? min(n32, icap) : n32, nw32 = idle ? nsp * nfree : nbl * WPB;
            const PairCoef<T> qv = coef_vv(p), qw = coef_vw(p);
            const bool fpx = sizeof(T) == 4 && p.bc[0] == BC_PERIODIC, fpy = sizeof(T) == 4 && p.bc[1] == BC_PERIODIC,
                       fpz = sizeof(T) == 4 && p.bc[2] == BC_PERIODIC;
            // a warp of a particle block that holds no lane group keeps its list's head in the group's carry registers
            // (the warp's first lane group has its lowest slot number: warp-uniform)
            const bool wcarry = cyon && !idle && !(nsp * GPB + (int)(threadIdx.x >> 5) * nbl + b < nh);
            for (int h = h0; h < hlim; h += nw32) {
                const bool first = h == h0, kept = wcarry && first && cy.hvalid;
                int i, raw, j[4];
                T vx = T(0), vy = T(0), vz = T(0);
                if (kept) {
                    i = cy.hi; raw = cy.hraw; vx = cy.hvx; vy = cy.hvy; vz = cy.hvz;
#pragma unroll
                    for (int u = 0; u < 4; ++u) j[u] = cy.hj[u];
                } else {
                    const int top = p.nv - 1 - h;
                    i = v.cell[top]; raw = v.slot[top];
                    const int nv0 = vl_nvv(raw), n0 = nv0 + vl_nvw(raw);
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int k = lane + 32 * u;
                        j[u] = k < n0 ? v.nbr[vl_base(i, VL_MAXN) + (k < nv0 ? k : k + VL_MAXN - n0) * VL_LS] : -1;
                    }
                    if (lane == 0) { vx = s.vx[i]; vy = s.vy[i]; vz = s.vz[i]; }
                }
                const int nvv = vl_nvv(raw);
                Vec4<T> rj[4];
                const Vec4<T> ri = rcur[i];
                vx = lam * vx; vy = lam * vy; vz = lam * vz;
#pragma unroll
                for (int u = 0; u < 4; ++u) rj[u] = rcur[max(j[u], 0)];
                Acc<T, false> a;
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const T dx = fpx ? fold(ri.x, rj[u].x, p.L[0], T(0.5) * p.L[0]) : ri.x - rj[u].x;
                    const T dy = fpy ? fold(ri.y, rj[u].y, p.L[1], T(0.5) * p.L[1]) : ri.y - rj[u].y;
                    const T dz = fpz ? fold(ri.z, rj[u].z, p.L[2], T(0.5) * p.L[2]) : ri.z - rj[u].z;
                    const bool wall = lane + 32 * u >= nvv;
                    PairCoef<T> qq;
                    qq.rc2 = qv.rc2; qq.c12 = wall ? qw.c12 : qv.c12; qq.c6 = wall ? qw.c6 : qv.c6;
                    pair_term_nb<T, false>(qq, j[u] >= 0, dx, dy, dz, a);
                }
                T fx = a.fx, fy = a.fy, fz = a.fz;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    fx += __shfl_xor_sync(0xffffffffu, fx, o);
                    fy += __shfl_xor_sync(0xffffffffu, fy, o);
                    fz += __shfl_xor_sync(0xffffffffu, fz, o);
                }
                if (lane == 0) {
                    if (!drift) { v.f.fx[i] = fx; v.f.fy[i] = fy; v.f.fz[i] = fz; }
                    Vec4<T> rn = ri;
                    integrate(i, ri, vx, vy, vz, fx, fy, fz, rn, vl_face(raw));
                }
                if (wcarry && first) {
                    cy.hi = i; cy.hraw = raw; cy.hvx = vx; cy.hvy = vy; cy.hvz = vz;
#pragma unroll
                    for (int u = 0; u < 4; ++u) cy.hj[u] = j[u];
                    cy.hvalid = drift;
                }
            }
        }
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
                for (int u = 0; u < 4; ++u) {
                    const int k = sub + VL_GROUP * u, nv0 = vl_nvv(raw), n0 = nv0 + vl_nvw(raw);
                    j0[u] = v.nbr[vl_base(i, VL_MAXN) + (k < nv0 || k >= n0 ? k : k + VL_MAXN - n0) * VL_LS];
                }
                if (sub == 0) { vx = s.vx[i]; vy = s.vy[i]; vz = s.vz[i]; }
            }
            const Vec4<T> ri = rcur[i];
            vx = lam * vx; vy = lam * vy; vz = lam * vz;
            Acc<T, false> a;
            const int nvv = vl_nvv(raw), n = nvv + vl_nvw(raw);
            const bool fold = sizeof(T) == 4 && __any_sync(__activemask(), vl_face(raw) != 0);
            if (fold) list_loop_group<T, true>(p, v.nbr + vl_base(i, VL_MAXN), nvv, n, sub, rcur, ri, j0, a);
            else list_loop_group<T, false>(p, v.nbr + vl_base(i, VL_MAXN), nvv, n, sub, rcur, ri, j0, a);
            T fx = a.fx, fy = a.fy, fz = a.fz;
#pragma unroll
            for (int o = 1; o < VL_GROUP; o <<= 1) {
                fx += __shfl_xor_sync(gmask, fx, o);
                fy += __shfl_xor_sync(gmask, fy, o);
                fz += __shfl_xor_sync(gmask, fz, o);
            }
            if (sub == 0) {
                if (!drift) { v.f.fx[i] = fx; v.f.fy[i] = fy; v.f.fz[i] = fz; }
                Vec4<T> rn = ri;
                integrate(i, ri, vx, vy, vz, fx, fy, fz, rn, vl_face(raw));
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
                                           bool kick, bool drift, bool& want, int gtid, int gthreads, int hp,
                                           T lam = T(1), double* ksum = nullptr)
{
    Carry<T> none;
    phase_step<T>(p, v, c, cv, force, kick, drift, want, gtid, gthreads, hp, lam, ksum, none, false);
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
        if (v.nprune > 0) v.wo[i] = T(0);                // paths since THIS full rebuild (any order: every entry is cleared)
        int cx, cy, cz;
        const int ci = cell_index(p, ri.x, ri.y, ri.z, cx, cy, cz);
        v.cell[i] = ci;
        v.slot[i] = atomicAdd(&v.count[ci], 1);
    }
}

__device__ __forceinline__ int block_sum_int(int x, int* ws)
{
    x = warp_sum(x);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = x;
    __syncthreads();
    int a = 0;
#pragma unroll
    for (int k = 0; k < VL_THREADS / 32; ++k) a += ws[k];
    return a;
}

// R2: exclusive scan of the counts in ONE phase, tiles strided over the blocks.  Pass A: a block sums each of its
// tiles and publishes (generation, sum) as one 64-bit word.  Pass B: the offset of a tile is the sum of the published
// sums before it -- read with relaxed loads, spinning while a word still carries an older generation (every block
// publishes all its sums before it waits for any, so nobody waits for a waiter) -- then a warp-shuffle scan inside the
// tile.  No second phase and no same-address atomics: 2048 warp atomics on the 21 tile sums of config 2 cost 10 us
// when tried in the bin phase (profiles/r02_k_md_run.md).  blockDim.x must equal VL_THREADS.
__device__ __forceinline__ void phase_scan(const int* __restrict__ count, int n, unsigned long long* __restrict__ tile_agg,
                                           unsigned int gen, int* __restrict__ start)
{
    __shared__ int ws[VL_THREADS / 32];
    const int tiles = (n + VS_TILE - 1) / VS_TILE;
    for (int t = blockIdx.x; t < tiles; t += gridDim.x) {
        const int base = t * VS_TILE + threadIdx.x * VS_ITEMS;
        int s = 0;
#pragma unroll
        for (int k = 0; k < VS_ITEMS; ++k) s += base + k < n ? count[base + k] : 0;
        const int sum = block_sum_int(s, ws);
        if (threadIdx.x == 0) {
            const unsigned long long word = ((unsigned long long)gen << 32) | (unsigned int)sum;
            asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(tile_agg + t), "l"(word) : "memory");
        }
    }
    for (int t = blockIdx.x; t < tiles; t += gridDim.x) {
        const int base = t * VS_TILE + threadIdx.x * VS_ITEMS;
        int val[VS_ITEMS];
        int s = 0;
#pragma unroll
        for (int k = 0; k < VS_ITEMS; ++k) {
            val[k] = base + k < n ? count[base + k] : 0;
            s += val[k];
        }
        int off = 0;
        for (int k = threadIdx.x; k < t; k += VL_THREADS) {
            unsigned long long word;
            do {
                asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(word) : "l"(tile_agg + k) : "memory");
            } while ((unsigned int)(word >> 32) != gen);
            off += (int)(unsigned int)word;
        }
        off = block_sum_int(off, ws);
        const int incl = warp_incl_scan(s);
        __syncthreads();
        if ((threadIdx.x & 31) == 31) ws[threadIdx.x >> 5] = incl;
        __syncthreads();
        int wofs = 0;
        for (int k = 0; k < (int)(threadIdx.x >> 5); ++k) wofs += ws[k];
        int run = off + wofs + incl - s;
#pragma unroll
        for (int k = 0; k < VS_ITEMS; ++k) {
            if (base + k < n) start[base + k] = run;     // counts are cleared in the list-build phase
            run += val[k];
        }
        if (base <= n - 1 && n - 1 < base + VS_ITEMS) start[n] = run;
        __syncthreads();
    }
}

// R3: scatter into cell order: positions c -> c^1 (plus their fp32 shadow), velocities / ids cv -> cv^1.
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
        const Vec4<T> ri = ra[i];
        rb[d] = ri;
        if (sizeof(T) == 8) v.r32[d] = F4{(float)ri.x, (float)ri.y, (float)ri.z, 0.f};
        b.vx[d] = a.vx[i]; b.vy[d] = a.vy[i]; b.vz[d] = a.vz[i];
        b.id[d] = a.id[i];
    }
}

template <typename T>
__device__ __forceinline__ int face_code(const Params<T>& p, int cx, int cy, int cz)
{
    int face = 0;
    if (p.bc[0] == BC_PERIODIC) face |= cx == 0 ? 1 : (cx == p.nc[0] - 1 ? 2 : 0);
    if (p.bc[1] == BC_PERIODIC) face |= (cy == 0 ? 1 : (cy == p.nc[1] - 1 ? 2 : 0)) << 2;
    if (p.bc[2] == BC_PERIODIC) face |= (cz == 0 ? 1 : (cz == p.nc[2] - 1 ? 2 : 0)) << 4;
    return face;
}

// End of a particle's list build: the ncnt word, the heavy registries (counter set hp), overflow, its ghost copies.
template <typename T>
__device__ __forceinline__ void finish_list(const Params<T>& p, const Verlet<T>& v, Vec4<T>* __restrict__ r, int i,
                                            const Vec4<T>& ri, int nvv, int nvw, int face, int hcap, int hcap32, int hp,
                                            bool ghosts = true)
{
    const int n = nvv + nvw;
    int raw = min(nvv, VL_MAXN) | (min(nvw, VL_MAXN) << VL_NVW_SHIFT) | (face << VL_FACE_SHIFT);
    if (n > VL_MAXN) { v.flags[VF_OVERFLOW] = 1; raw = face << VL_FACE_SHIFT; }      // reported by the host; the list is not used
    // a long list goes to a lane group (a very long one to a warp) while the idle blocks have some left; the counters
    // keep the demand and the host sizes the next launch by it; `cell` and `slot` are free until the next rebuild
    // (what its own thread would pay is batches, and the two kinds of entries are batched separately: six vapor and six
    // wall entries cost four batches where twelve vapor entries cost three)
    else if (n > v.heavy_t || ((nvv + VL_BATCH - 1) / VL_BATCH + (nvw + VL_BATCH - 1) / VL_BATCH) * VL_BATCH > v.heavy_t + VL_BATCH - 1) {
        bool placed = false;
        if (n > VL_WARP_T && hcap32 > 0) {
            const int h = atomicAdd(v.flags + VF_NHEAVY32 + hp, 1);
            placed = h < hcap32;
            if (placed) { raw |= VL_HEAVY; v.cell[p.nv - 1 - h] = i; v.slot[p.nv - 1 - h] = raw; }
        }
        if (!placed) {                                   // no warp left: four lanes are still better than one
            const int h = atomicAdd(v.flags + VF_NHEAVY + hp, 1);
            if (h < hcap) { raw |= VL_HEAVY; v.cell[h] = i; v.slot[h] = raw; }
        }
    }
    v.ncnt[i] = raw;
    if (sizeof(T) == 8 && face && ghosts) write_ghosts(p, v, r, i, ri, face);
}

// finish_list for a CONVERGED warp (every lane calls it, `live` lanes have a particle): one atomic per warp and registry
// instead of one per long list -- particles with long lists sit together (a film, a cluster), and a burst of ~2,000
// same-address atomics with a return value at the end of a short phase is what the phase then waits for.
template <typename T>
__device__ __forceinline__ void finish_list_warp(const Params<T>& p, const Verlet<T>& v, int i, bool live, int nvv, int nvw, int face,
                                                 int hcap, int hcap32, int hp)
{
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const int n = nvv + nvw;
    int raw = min(nvv, VL_MAXN) | (min(nvw, VL_MAXN) << VL_NVW_SHIFT) | (face << VL_FACE_SHIFT);
    const bool over = live && n > VL_MAXN;
    if (over) { v.flags[VF_OVERFLOW] = 1; raw = face << VL_FACE_SHIFT; }
    const bool heavy = live && !over &&
                       (n > v.heavy_t || ((nvv + VL_BATCH - 1) / VL_BATCH + (nvw + VL_BATCH - 1) / VL_BATCH) * VL_BATCH > v.heavy_t + VL_BATCH - 1);
    const bool want32 = heavy && n > VL_WARP_T && hcap32 > 0;
    const unsigned m32 = __ballot_sync(0xffffffffu, want32);
    int b32 = 0;
    if (lane == 0 && m32) b32 = atomicAdd(v.flags + VF_NHEAVY32 + hp, __popc(m32));
    b32 = __shfl_sync(0xffffffffu, b32, 0);
    bool placed = false;
    if (want32) {
        const int h = b32 + __popc(m32 & lt);
        placed = h < hcap32;
        if (placed) { raw |= VL_HEAVY; v.cell[p.nv - 1 - h] = i; v.slot[p.nv - 1 - h] = raw; }
    }
    const bool want4 = heavy && !placed;
    const unsigned m4 = __ballot_sync(0xffffffffu, want4);
    int b4 = 0;
    if (lane == 0 && m4) b4 = atomicAdd(v.flags + VF_NHEAVY + hp, __popc(m4));
    b4 = __shfl_sync(0xffffffffu, b4, 0);
    if (want4) {
        const int h = b4 + __popc(m4 & lt);
        if (h < hcap) { raw |= VL_HEAVY; v.cell[h] = i; v.slot[h] = raw; }
    }
    if (live) v.ncnt[i] = raw;
}

// R4: neighbour list from the cell list (a3's cell traversal, cached): every j within r_c + skin of i, vapor entries from
// slot 0 up, wall entries from the top slot down.  ROWS = 3^(d-1) lanes cooperate on one particle: lane `row` walks the
// cell row (cy + ky, cz + kz) -- its three cells are one contiguous range of the cell-ordered arrays, plus the wrapped
// cell at a periodic x face -- eight candidate loads in flight at a time, and appends its hits through two
// shared-memory counters.  The periodic image is applied once per row / segment as a shift of r_i, and an entry records
// the image block of the ghost copy the time loop will read (fp64; fp32 mode stores plain indices and folds).  The
// distance filter runs in FP32 on the fp32 shadow of the positions with a threshold inflated by the rounding involved: the
// list is a superset of the pairs within r_c + skin, which is all the exactness argument needs.  Positions are wrapped here.
//
// Why this shape (profiles/r02_k_md_run.md): vapor at density 0.05 and T* = 1 condenses, so a few hundred particles sit in
// clusters and films with ten times the candidates of the rest, and the phase ends when the slowest warp does.  Units of
// work whose cost grows with the SQUARE of the local density -- a warp per block of cells, candidates in a tile: measured
// at 45-60 us -- lose to this one, where a particle's candidates are spread over nine lanes and three particles share a
// warp: its cost is linear in the density (39 us in round 1, in FP64 with folds).
// One range of candidates for particle i.  cnt[0], cnt[1]: inner / outer counters of the section (shared memory).
// Per batch of NB candidates a lane turns its hits into two bit masks, reserves their slots with ONE shared-memory atomic
// per list, and stores them in a loop that runs as long as the lane with the most hits needs (3-4 trips for 8 candidates).
// The obvious form -- test, atomic and store inside one `if` per candidate -- executes that hit path once per candidate
// slot, because among the 27 active lanes some lane nearly always hits: it was half of the build's 10,300 instructions per
// warp (ncu, profiles/r02_k_md_run.md).  (Eight predicated store sequences per batch instead of the loop were no faster.)
template <typename T, bool OUTER>
__device__ __forceinline__ void list_range(const Verlet<T>& v, const F4* __restrict__ q, int jb, int je, int skip, float xe, float ye,
                                           float ze, int e0, int i, int* cnt, bool up)
{
    constexpr int NB = 8;                                                // a cell row rarely holds more
    const float rl2 = v.rl2f, rl2o = v.rl2f_out;
    int* __restrict__ il = v.nbr + vl_base(i, VL_MAXN);
    int* __restrict__ ol = OUTER ? v.onbr + vl_base(i, VL_MAXO) : nullptr;
    for (int j0 = jb; j0 < je; j0 += NB) {
        F4 rj[NB];
#pragma unroll
        for (int u = 0; u < NB; ++u) rj[u] = q[min(j0 + u, je - 1)];     // NB loads in flight
        unsigned mi = 0u, mo = 0u;
#pragma unroll
        for (int u = 0; u < NB; ++u) {
            const float dx = xe - rj[u].x, dy = ye - rj[u].y, dz = ze - rj[u].z;
            const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            const unsigned ok = (unsigned)(j0 + u < je) & (unsigned)(j0 + u != skip);
            mi |= (ok & (unsigned)(r2 < rl2)) << u;
            if (OUTER) mo |= (ok & (unsigned)(r2 < rl2o)) << u;
        }
        if (OUTER && mo) {
            int k = atomicAdd(cnt + 1, __popc(mo));
            do {
                const int u = __ffs(mo) - 1;
                mo &= mo - 1u;
                if (k < VL_MAXO) ol[(up ? k : VL_MAXO - 1 - k) * VL_LS] = e0 + j0 + u;
                ++k;
            } while (mo);
        }
        if (mi) {
            int k = atomicAdd(cnt, __popc(mi));
            do {
                const int u = __ffs(mi) - 1;
                mi &= mi - 1u;
                if (k < VL_MAXN) il[(up ? k : VL_MAXN - 1 - k) * VL_LS] = e0 + j0 + u;
                ++k;
            } while (mi);
        }
    }
}

// OUTER: the cells have side >= r_c + outer skin and every hit also goes to the outer list (two-level list).
template <typename T, int ROWS, bool OUTER>
__device__ __forceinline__ void phase_build(const Params<T>& p, const Verlet<T>& v, int c, int gtid, int gthreads, int hcap,
                                            int hcap32, int hp)
{
    constexpr bool GHOSTS = sizeof(T) == 8;
    constexpr int PPW = 32 / ROWS;                       // particles per warp
    __shared__ int s_cv[(VL_THREADS / 32) * PPW][2], s_cw[(VL_THREADS / 32) * PPW][2];
    Vec4<T>* __restrict__ r = v.st[c].r;
    const F4* __restrict__ q = GHOSTS ? v.r32 : reinterpret_cast<const F4*>(r);
    const int nx = p.nc[0], ny = p.nc[1], nz = p.nc[2];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int pl = lane / ROWS, row = lane - pl * ROWS;
    const int warp = gtid >> 5, nwarps = gthreads >> 5;
    int* cv = s_cv[wib * PPW + min(pl, PPW - 1)];
    int* cw = s_cw[wib * PPW + min(pl, PPW - 1)];
    const int istride = GHOSTS ? v.ntot : 0;
    for (int base = warp * PPW; base < p.nv; base += nwarps * PPW) {
        const int i = base + pl;
        const bool active = pl < PPW && i < p.nv;
        if (active && row == 0) { cv[0] = cv[1] = 0; cw[0] = cw[1] = 0; }
        __syncwarp();
        Vec4<T> ri = {T(0), T(0), T(0), T(0)};
        int face = 0;
        if (active) {
            ri = r[i];
            int cx, cy, cz;
            const int ci = cell_index(p, ri.x, ri.y, ri.z, cx, cy, cz);
            face = face_code(p, cx, cy, cz);
            int qy = cy + row % 3 - 1, qz = cz + (ROWS == 9 ? row / 3 - 1 : 0);
            bool ok = true;
            float ye = (float)ri.y, ze = (float)ri.z;
            int img = 0;
            // r_i in the first cell looking at the last one: the neighbour's image is at r_j - L, i.e. r_i + L
            if (qz < 0) { ok = p.bc[2] == BC_PERIODIC; qz += nz; ze += (float)p.L[2]; img |= 4; }
            else if (qz >= nz) { ok = p.bc[2] == BC_PERIODIC; qz -= nz; ze -= (float)p.L[2]; img |= 4; }
            if (qy < 0) { ok = ok && p.bc[1] == BC_PERIODIC; qy += ny; ye += (float)p.L[1]; img |= 2; }
            else if (qy >= ny) { ok = ok && p.bc[1] == BC_PERIODIC; qy -= ny; ye -= (float)p.L[1]; img |= 2; }
            if (ok) {
                const int x0 = max(cx - 1, 0), x1 = min(cx + 1, nx - 1);
                int xw = -1;
                float xe = (float)ri.x, xe2 = xe;
                if (p.bc[0] == BC_PERIODIC) { if (cx == 0) { xw = nx - 1; xe2 += (float)p.L[0]; } else if (cx == nx - 1) { xw = 0; xe2 -= (float)p.L[0]; } }
                const int rowc = (qz * ny + qy) * nx;
                const bool do_wall = p.nw > 0 && v.wnear[ci];
                // all cell-start loads first (independent), then the particle loops
                const int jb = v.start[rowc + x0], je = v.start[rowc + x1 + 1];
                int jb2 = 0, je2 = 0, wb = 0, we = 0, wb2 = 0, we2 = 0;
                if (xw >= 0) { jb2 = v.start[rowc + xw]; je2 = v.start[rowc + xw + 1]; }
                if (do_wall) {
                    wb = v.wstart[rowc + x0]; we = v.wstart[rowc + x1 + 1];
                    if (xw >= 0) { wb2 = v.wstart[rowc + xw]; we2 = v.wstart[rowc + xw + 1]; }
                }
                list_range<T, OUTER>(v, q, jb, je, img ? -1 : i, xe, ye, ze, img * istride, i, cv, true);
                list_range<T, OUTER>(v, q, jb2, je2, -1, xe2, ye, ze, (img | 1) * istride, i, cv, true);
                list_range<T, OUTER>(v, q + p.nv, wb, we, -1, xe, ye, ze, img * istride + p.nv, i, cw, false);
                list_range<T, OUTER>(v, q + p.nv, wb2, we2, -1, xe2, ye, ze, (img | 1) * istride + p.nv, i, cw, false);
            }
        }
        __syncwarp();
        if (active && row == 0) {
            finish_list(p, v, r, i, ri, cv[0], cw[0], face, hcap, hcap32, hp);
            if (OUTER) {
                const int ov = cv[1], ow = cw[1];
                int word = min(ov, VL_MAXO) | (min(ow, VL_MAXO) << VO_W_SHIFT) | (face << VO_FACE_SHIFT);
                if (ov + ow > VL_MAXO) v.flags[VF_OUTER_BAD] = 1;            // not an error: no pruning from this list
                else if (ov + ow > VO_HEAVY_T) { word |= VO_HEAVY; v.oheavy[atomicAdd(v.flags + VF_NOHEAVY, 1)] = i; }
                v.ocnt[i] = word;
            }
        }
        __syncwarp();
    }
}

// R5, two-level list (the verdict's "take the rebuild off the critical path"): between two full
// rebuilds the r_c + skin list is PRUNED from the outer list (every j within r_c + outer skin at the last full rebuild)
// instead of being rebuilt from the cells: no bin, no scan, no scatter, no cell walk, ~17 distance tests per particle
// instead of ~55 candidates -- one phase and one barrier, in the particle order of the last full rebuild.
// Exactness: a pair within r_c + skin now was within r_c + outer skin at the full rebuild provided neither particle's
// path since then exceeds outer_lim = (outer skin - skin) / 2.  The prune accumulates every particle's path (wo += w,
// w = 0) and checks exactly that; if any particle violates it the caller discards the prune and runs a full rebuild
// (the host sizes the outer skin so that this is rare: (nprune + 1) skins plus a margin for the step that crosses).
// Tests are made on the positions themselves (T), entries keep their image codes; fp32 mode folds.  Particles with a long
// outer list (VO_HEAVY: condensed regions) are pruned by a whole warp each, spread over all warps of the grid.
// Returns: this thread saw a path beyond outer_lim.
template <typename T, int NB>
__device__ __forceinline__ bool phase_prune(const Params<T>& p, const Verlet<T>& v, int c, int gtid, int gthreads, int hcap,
                                            int hcap32, int hp)
{
    constexpr bool FOLD = sizeof(T) == 4;
    Vec4<T>* __restrict__ r = v.st[c].r;
    const bool px = FOLD && p.bc[0] == BC_PERIODIC, py = FOLD && p.bc[1] == BC_PERIODIC, pz = FOLD && p.bc[2] == BC_PERIODIC;
    const T rl2 = v.rl2_prune;
    bool bad = false;
#ifdef MD_DIAGNOSTICS
    const unsigned long long t_in = now_ns();
#endif
    auto dist2 = [&](const Vec4<T>& ri, const Vec4<T>& rj) {
        const T dx = px ? fold(ri.x, rj.x, p.L[0], T(0.5) * p.L[0]) : ri.x - rj.x;
        const T dy = py ? fold(ri.y, rj.y, p.L[1], T(0.5) * p.L[1]) : ri.y - rj.y;
        const T dz = pz ? fold(ri.z, rj.z, p.L[2], T(0.5) * p.L[2]) : ri.z - rj.z;
        return fma_(dz, dz, fma_(dy, dy, dx * dx));
    };
    auto close = [&](int i, const Vec4<T>& ri, int nvv, int nvw, int face) {
        const T wsum = v.wo[i] + ri.w;                   // path since the full rebuild
        v.wo[i] = wsum;
        if (wsum > v.outer_lim) bad = true;
        r[i].w = T(0);                                   // path since this list event
        finish_list(p, v, r, i, ri, nvv, nvw, face, hcap, hcap32, hp, false);
    };
    // ---- one thread per particle (the warp stays converged: lanes without work run with empty lists)
    for (int i0 = gtid - (int)(threadIdx.x & 31); i0 < p.nv; i0 += gthreads) {
        const int i = i0 + (int)(threadIdx.x & 31);
        const bool inrange = i < p.nv;
        int olv[NB];                                     // issued together with the count word
        {
            const int* __restrict__ o0 = v.onbr + vl_base(i, VL_MAXO);
#pragma unroll
            for (int u = 0; u < NB; ++u) olv[u] = o0[u * VL_LS];
        }
        const int word = inrange ? v.ocnt[i] : VO_HEAVY;
        const bool live = !(word & VO_HEAVY);
        const Vec4<T> ri = r[inrange ? i : 0];
        const T wold = inrange ? v.wo[i] : T(0);         // issued early
        const int ov = live ? word & VO_MASK : 0, ow = live ? (word >> VO_W_SHIFT) & VO_MASK : 0;
        const int* __restrict__ ol = v.onbr + vl_base(i, VL_MAXO);
        int* __restrict__ il = v.nbr + vl_base(i, VL_MAXN);
        int cnt[2] = {0, 0};
#pragma unroll
        for (int sec = 0; sec < 2; ++sec) {              // vapor entries from slot 0 up, wall entries from the top slot down
            const int ne = sec ? ow : ov;
            int en[NB];
            if (sec == 0) {                              // the first vapor entries do not wait for the count (the rows exist)
#pragma unroll
                for (int u = 0; u < NB; ++u) en[u] = olv[u];
#pragma unroll
                for (int u = 0; u < NB; ++u) en[u] = u < ne ? en[u] : -1;
            } else {
#pragma unroll
                for (int u = 0; u < NB; ++u) en[u] = u < ne ? ol[(VL_MAXO - 1 - u) * VL_LS] : -1;
            }
            for (int k = 0; k < ne; k += NB) {
                int e[NB];
                Vec4<T> rj[NB];
#pragma unroll
                for (int u = 0; u < NB; ++u) { e[u] = en[u]; rj[u] = r[max(e[u], 0)]; }
#pragma unroll
                for (int u = 0; u < NB; ++u) {
                    const int kk = k + NB + u;
                    en[u] = kk < ne ? ol[(sec ? VL_MAXO - 1 - kk : kk) * VL_LS] : -1;      // next batch
                }
                // all NB distances first -- independent FP64 chains, interleaved -- then the appends: written as one loop the
                // compiler made every test a divergent branch around its own dependent chain (56 instructions per entry)
                T r2[NB];
#pragma unroll
                for (int u = 0; u < NB; ++u) r2[u] = dist2(ri, rj[u]);
#pragma unroll
                for (int u = 0; u < NB; ++u) {
                    const int hit = (int)(e[u] >= 0) & (int)(r2[u] < rl2);
                    const int at = sec ? VL_MAXN - 1 - cnt[sec] : cnt[sec];
                    if (hit & (int)(cnt[sec] < VL_MAXN)) il[at * VL_LS] = e[u];
                    cnt[sec] += hit;
                }
            }
        }
        if (live) {
            const T wsum = wold + ri.w;                  // path since the full rebuild
            v.wo[i] = wsum;
            if (wsum > v.outer_lim) bad = true;
            r[i].w = T(0);                               // path since this list event
        }
        finish_list_warp(p, v, i, live, cnt[0], cnt[1], (word >> VO_FACE_SHIFT) & VL_FACE_MASK, hcap, hcap32, hp);
    }
#ifdef MD_DIAGNOSTICS
    const unsigned long long tl = now_ns();
#endif
    // ---- one warp per particle with a long outer list
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const int noh = v.flags[VF_NOHEAVY];
    // the warps of the blocks past the last particle have no list of their own to prune: they take these first, so that the
    // long lists run beside the short ones instead of after them
    const int nbl = min((int)gridDim.x, (p.nv + VL_THREADS - 1) / VL_THREADS), nidlew = ((int)gridDim.x - nbl) * (VL_THREADS / 32);
    const int widx = (int)blockIdx.x >= nbl ? (gtid >> 5) - nbl * (VL_THREADS / 32) : nidlew + (gtid >> 5);
    for (int h = widx; h < noh; h += gthreads >> 5) {
        const int i = v.oheavy[h];
        const int word = v.ocnt[i];
        const Vec4<T> ri = r[i];
        const int ov = word & VO_MASK, ow = (word >> VO_W_SHIFT) & VO_MASK;
        const int* __restrict__ ol = v.onbr + vl_base(i, VL_MAXO);
        int* __restrict__ il = v.nbr + vl_base(i, VL_MAXN);
        int cnt[2] = {0, 0};
#pragma unroll
        for (int sec = 0; sec < 2; ++sec) {
            const int ne = sec ? ow : ov;
            constexpr int NI = 4;                        // 128 entries per round: all index loads, then all position loads, in flight
            for (int k0 = 0; k0 < ne; k0 += 32 * NI) {
                int e[NI];
                Vec4<T> rj[NI];
#pragma unroll
                for (int u = 0; u < NI; ++u) {
                    const int k = k0 + 32 * u + lane;
                    e[u] = k < ne ? ol[(sec ? VL_MAXO - 1 - k : k) * VL_LS] : -1;
                }
#pragma unroll
                for (int u = 0; u < NI; ++u) rj[u] = r[max(e[u], 0)];
                T r2[NI];
#pragma unroll
                for (int u = 0; u < NI; ++u) r2[u] = dist2(ri, rj[u]);
#pragma unroll
                for (int u = 0; u < NI; ++u) {
                    const bool hit = (e[u] >= 0) & (r2[u] < rl2);
                    const unsigned m = __ballot_sync(0xffffffffu, hit);
                    const int pos = cnt[sec] + __popc(m & lt);
                    if (hit && pos < VL_MAXN) il[(sec ? VL_MAXN - 1 - pos : pos) * VL_LS] = e[u];
                    cnt[sec] += __popc(m);
                }
            }
        }
        if (lane == 0) close(i, ri, cnt[0], cnt[1], (word >> VO_FACE_SHIFT) & VL_FACE_MASK);
        __syncwarp();
    }
#ifdef MD_DIAGNOSTICS
    if (v.dbg && lane == 0) {          // per warp: ns in the two parts, summed over prunes; [2]: particles pruned by warps
        atomicAdd(v.dbg + 4096 + 2 * ((gtid >> 5) & 1023), tl - t_in);
        atomicAdd(v.dbg + 4097 + 2 * ((gtid >> 5) & 1023), now_ns() - tl);
        if (gtid == 0) v.dbg[7000] += noh;
    }
#endif
    return bad;
}

// ---- the persistent time loop ---------------------------------------------------------------------
// md_step(n): phase(stored f; kick + drift), then n - 1 fused phases (force; kick; kick + drift), then
// phase(force; kick): n + 1 phases and n grid barriers for n steps, plus 4 barriers per rebuild.
// force_rebuild (md_create): bin + build the list first, then evaluate f(0).
// MINB = resident blocks per SM the register budget is sized for: 2 (up to 128 registers, the latency-bound
// sizes that fit one wave) or 3 (more warps to hide HBM latency once the state no longer fits in L2).
template <typename T, int ROWS, int MINB>
__global__ void __launch_bounds__(VL_THREADS, (MINB * 256) / VL_THREADS) k_md_run(Params<T> p, Verlet<T> v, long long n_steps, int force_rebuild)
{
    __shared__ unsigned long long s_times[10];
    GridBarrier bar_seq;
    const bool thermo = p.thermo_rate > 0.0;
    const int gtid = blockIdx.x * blockDim.x + threadIdx.x;
    const int gthreads = gridDim.x * blockDim.x;
    int c = v.flags[VF_CUR], cv = v.flags[VF_CURV];
    bool rebuild = force_rebuild != 0;
    Carry<T> carry;
    const bool cyon = MINB == 2 && v.carry && !thermo && gthreads >= p.nv;      // (the 3-blocks-per-SM variant serves N > one wave)
    // lane groups in the blocks past the last particle (none once the particles fill the grid)
    const int nidle = max((int)gridDim.x - (p.nv + VL_THREADS - 1) / VL_THREADS, 0);
    // whole-warp lists: VL_WARP_ROUNDS per warp of the idle blocks, one per warp of the particle blocks
    const int hcap = nidle * (VL_THREADS / VL_GROUP),
              hcap32 = (nidle * VL_WARP_ROUNDS + ((int)gridDim.x - nidle)) * (VL_THREADS / 32);
    if (gtid == 0)
        for (int k = 0; k < 10; ++k) s_times[k] = 0;
    unsigned long long t0 = gtid == 0 ? now_ns() : 0ull, t1;
    int hp = v.flags[VF_HPAR];          // which set of heavy-list counters the step phases read
    int since_full = 1 << 30;           // prunes since the last full rebuild (unknown at launch: the first event is a full one
                                        // unless the previous launch left a usable outer list, see below)
    if (v.nprune > 0 && !force_rebuild) since_full = v.flags[VF_NPRUNE + 1];
    for (long long s = 0;; ++s) {
        if (rebuild) {
            unsigned long long u0 = gtid == 0 ? now_ns() : 0ull, u1;
            const int hw = hp ^ 1;                                       // the counter set this list event fills
            if (gtid == 0) { v.flags[VF_HCAP] = hcap; v.flags[VF_HCAP32] = hcap32; }
            bool full = force_rebuild || since_full >= v.nprune || *(volatile int*)(v.flags + VF_OUTER_BAD) != 0;
            if (!full) {
                const bool bad = phase_prune<T, MINB == 2 ? 8 : 4>(p, v, c, gtid, gthreads, hcap, hcap32, hw);
                if (gtid == 0) v.flags[VF_NPRUNE] += 1;
                full = grid_barrier(v.bar, bar_seq, bad);                // a path beyond outer_lim: the prune is void
                ++since_full;
                if (gtid == 0) { t1 = now_ns(); s_times[2] += t1 - t0; s_times[8] += t1 - t0; t0 = t1; u0 = t1; }
                if (full && gtid == 0) { v.flags[VF_NHEAVY + hw] = 0; v.flags[VF_NHEAVY32 + hw] = 0; }    // refilled below
            }
            if (full) {
                if (gtid == 0) v.flags[VF_NOHEAVY] = 0;
                phase_bin<T>(p, v, c, gtid, gthreads);
                grid_barrier(v.bar, bar_seq);
                if (gtid == 0) { u1 = now_ns(); s_times[4] += u1 - u0; u0 = u1; }
                phase_scan(v.count, p.ncell, v.tile_agg, (unsigned int)v.flags[VF_NREBUILD] + 1u, v.start);
                grid_barrier(v.bar, bar_seq);
                if (gtid == 0) { u1 = now_ns(); s_times[5] += u1 - u0; u0 = u1; }
                phase_scatter<T>(p, v, c, cv, gtid, gthreads);
                if (gtid == 0) v.flags[VF_OUTER_BAD] = 0;                // everybody has taken this event's decision by now
                grid_barrier(v.bar, bar_seq);
                if (gtid == 0) { u1 = now_ns(); s_times[6] += u1 - u0; u0 = u1; }
                c ^= 1; cv ^= 1;
                if (v.nprune > 0) phase_build<T, ROWS, true>(p, v, c, gtid, gthreads, hcap, hcap32, hw);
                else phase_build<T, ROWS, false>(p, v, c, gtid, gthreads, hcap, hcap32, hw);
                for (int q = gtid; q < p.ncell; q += gthreads) v.count[q] = 0;                  // for the next rebuild
                if (gtid == 0) v.flags[VF_NREBUILD] += 1;
                grid_barrier(v.bar, bar_seq);
                since_full = 0;
                if (gtid == 0) { t1 = now_ns(); s_times[2] += t1 - t0; t0 = t1; s_times[7] += t1 - u0; }
            }
            hp = hw;
            if (gtid == 0) { v.flags[VF_NHEAVY + (hp ^ 1)] = 0; v.flags[VF_NHEAVY32 + (hp ^ 1)] = 0; }   // the retired set, for the next event
            carry.valid = carry.hvalid = carry.nhvalid = false;          // new lists (and, after a full rebuild, a new particle order)
        }
        if (s == n_steps) break;
        bool want = false;                                   // this thread asks for a rebuild before the next step
        if (gtid == 0 && thermo) v.ksum[(s + 1) % 3] = 0.0;                                  // slot of step s + 1
#ifdef MD_DIAGNOSTICS
        unsigned long long dbg0 = 0;
        if (v.dbg) dbg0 = now_ns();
#endif
        if (!thermo || s == 0) {
            phase_step<T>(p, v, c, cv, s > 0, s > 0, true, want, gtid, gthreads, hp, T(1), nullptr, carry, cyon);
        } else {
            // with the thermostat lambda(t) needs K(t) of ALL particles before the next drift: the fused phase splits
            // into [F1 + F3 + K partial sums] | barrier | [F4 rescale + F2], one extra barrier per step
            phase_step<T>(p, v, c, cv, true, true, false, want, gtid, gthreads, hp, T(1), v.ksum + s % 3);
            grid_barrier(v.bar, bar_seq);
            const double lam = berendsen_lambda(*(volatile double*)(v.ksum + s % 3), p.thermo_rate, p.t_target, p.dof);
            phase_step<T>(p, v, c, cv, false, false, true, want, gtid, gthreads, hp, (T)lam);
        }
#ifdef MD_DIAGNOSTICS
        if (v.dbg && (threadIdx.x & 31) == 0) {
            const unsigned long long dt = now_ns() - dbg0;
            atomicAdd(v.dbg + (gtid >> 5), dt);
            atomicAdd(v.dbg + 8000 + min((int)(dt >> 10), 15), 1ull);       // histogram of warp-phase times, ~1 us bins
        }
#endif
        if (gtid == 0) { t1 = now_ns(); s_times[0] += t1 - t0; t0 = t1; }
        rebuild = grid_barrier(v.bar, bar_seq, want);       // some particle's path since the last rebuild exceeds skin / 2
        if (gtid == 0) { t1 = now_ns(); s_times[1] += t1 - t0; t0 = t1; }
        c ^= 1;
    }
    if (thermo && n_steps > 0) {
        double* ks = v.ksum + n_steps % 3;
        bool unused = false;
        phase_step<T>(p, v, c, cv, true, true, false, unused, gtid, gthreads, hp, T(1), ks);
        grid_barrier(v.bar, bar_seq);
        const double lam = berendsen_lambda(*(volatile double*)ks, p.thermo_rate, p.t_target, p.dof);
        phase_step<T>(p, v, c, cv, false, false, false, unused, gtid, gthreads, hp, (T)lam);      // F4 of the last step
    } else if (n_steps > 0 || force_rebuild) {
        bool unused = false;
        phase_step<T>(p, v, c, cv, true, n_steps > 0, false, unused, gtid, gthreads, hp);
    }
    if (gtid == 0) {
        v.flags[VF_CUR] = c; v.flags[VF_CURV] = cv;
        s_times[3] += now_ns() - t0;
        for (int k = 0; k < 10; ++k) v.times[k] += s_times[k];
        v.flags[VF_HPAR] = hp; v.flags[VF_NPRUNE + 1] = since_full;
    }
}

#ifdef MD_DIAGNOSTICS
// Diagnostics build only: the list-build phase as a kernel of its own, so that ncu can attribute its stalls.  It
// rebuilds the list from the current cell order, which is what the list already holds.
template <typename T, int ROWS>
__global__ void __launch_bounds__(VL_THREADS, 512 / VL_THREADS) k_dbg_build(Params<T> p, Verlet<T> v, int c)
{
    const int gtid = blockIdx.x * blockDim.x + threadIdx.x, gthreads = gridDim.x * blockDim.x;
    if (v.nprune > 0) phase_build<T, ROWS, true>(p, v, c, gtid, gthreads, v.flags[VF_HCAP], v.flags[VF_HCAP32], v.flags[VF_HPAR]);
    else phase_build<T, ROWS, false>(p, v, c, gtid, gthreads, v.flags[VF_HCAP], v.flags[VF_HCAP32], v.flags[VF_HPAR]);
}

// Diagnostics build only: the prune phase as a kernel of its own (valid at any time: it re-prunes from the outer list).
template <typename T>
__global__ void __launch_bounds__(VL_THREADS, 512 / VL_THREADS) k_dbg_prune(Params<T> p, Verlet<T> v, int c)
{
    phase_prune<T, 8>(p, v, c, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x, 0, 0, v.flags[VF_HPAR] ^ 1);
}

// Diagnostics build only: the force part of the step phase as a kernel of its own (recomputes f(t)).
template <typename T>
__global__ void __launch_bounds__(VL_THREADS, 512 / VL_THREADS) k_dbg_force(Params<T> p, Verlet<T> v, int c, int cv)
{
    bool unused = false;
    phase_step<T>(p, v, c, cv, true, false, false, unused, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x, v.flags[VF_HPAR]);
}
#endif

// Ghost copies of the wall particles (static, both position buffers), md_create only.
template <typename T>
__global__ void k_wall_ghosts(Params<T> p, Verlet<T> v)
{
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= p.nw) return;
    const Vec4<T> rw = v.st[0].r[p.nv + w];
    int cx, cy, cz;
    cell_index(p, rw.x, rw.y, rw.z, cx, cy, cz);
    int face = 0;
    if (p.bc[0] == BC_PERIODIC) face |= cx == 0 ? 1 : (cx == p.nc[0] - 1 ? 2 : 0);
    if (p.bc[1] == BC_PERIODIC) face |= (cy == 0 ? 1 : (cy == p.nc[1] - 1 ? 2 : 0)) << 2;
    if (p.bc[2] == BC_PERIODIC) face |= (cz == 0 ? 1 : (cz == p.nc[2] - 1 ? 2 : 0)) << 4;
    v.r32[p.nv + w] = F4{(float)rw.x, (float)rw.y, (float)rw.z, 0.f};
    if (face)
        for (int b = 0; b < 2; ++b) write_ghosts(p, v, v.st[b].r, p.nv + w, rw, face);
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
