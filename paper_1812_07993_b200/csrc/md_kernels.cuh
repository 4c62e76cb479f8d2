// md_kernels.cuh -- hand-written sm_100a kernels of the LJ pore-MD hot path.
// Steps a1-a5 of DESIGN.md; PAPER.md:57, :69-93 (kernels F1, F2, F3).
// 2D systems run with z = vz = fz = 0, one cell layer and bc[2] = BC_NONE, which
// leaves every r^2 = fma(dz, dz, fma(dy, dy, dx*dx)) bit-identical to the 2D form.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace md {

enum { BC_PERIODIC = 0, BC_REFLECT = 1, BC_NONE = 2 };

template <typename T>
struct Params {
    int nv, nw;
    T L[3], invL[3];
    int bc[3];
    int nc[3];
    int ncell;
    T inv_c[3];
    T rc2;
    T sig2_vv, e24_vv, e4_vv, uc_vv;
    T sig2_vw, e24_vw, e4_vw, uc_vw;
    T c12_vv, c6_vv, c12_vw, c6_vw;       // 48 eps sigma^12, 24 eps sigma^6: g = (c12 / r^6 - c6) / r^8 (time loop)
    T dt, hk; // hk = dt / (2 m)
    double mass;
    double thermo_rate, t_target, dof;   // Berendsen F4: dt / tau_B (0 = off), T_0, dim * n_vapor
    int prism, prism_axis;               // NEXT-3: geometric pore walls (closed faces reflect, +axis face open)
    T prism_c[3], prism_h[3];            // centre, half sizes (unused dimensions: c = 0, h = 1)
};

// Packed position: one 4-wide vector load per neighbour (w is spare; the cell path keeps the
// path length since the last re-bin there).
template <typename T>
struct alignas(4 * sizeof(T)) Vec4 {
    T x, y, z, w;
};

// Particle state (a0): positions packed (x, y, z, w), velocities SoA. One of two ping-pong
// buffers; id = caller's original index.
template <typename T>
struct State {
    Vec4<T>* r;
    T *vx, *vy, *vz;
    int* id;
};

template <typename T>
struct Force {
    T *fx, *fy, *fz;
};

// Per-particle energy-pass outputs (a5), always fp64.
struct EnergyOut {
    double *pe, *pew, *vir;
    int *cvv, *cvw;
};

template <typename T>
struct Walls {
    const Vec4<T>* r;         // sorted by cell
    const int* start;         // [ncell + 1]
    const uint8_t* near;      // [ncell]: any wall particle in the 3^d neighbourhood
};

__device__ __forceinline__ double rint_(double a) { return rint(a); }
__device__ __forceinline__ float rint_(float a) { return rintf(a); }
__device__ __forceinline__ double floor_(double a) { return floor(a); }
__device__ __forceinline__ float floor_(float a) { return floorf(a); }
__device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }

template <typename T>
__device__ __forceinline__ int cell_coord(T r, T inv_c, int n)
{
    int k = (int)(r * inv_c);
    return min(max(k, 0), n - 1);
}

template <typename T>
__device__ __forceinline__ int cell_index(const Params<T>& p, T x, T y, T z, int& cx, int& cy, int& cz)
{
    cx = cell_coord(x, p.inv_c[0], p.nc[0]);
    cy = cell_coord(y, p.inv_c[1], p.nc[1]);
    cz = cell_coord(z, p.inv_c[2], p.nc[2]);
    return (cz * p.nc[1] + cy) * p.nc[0] + cx;
}

// ---------------------------------------------------------------------------
// a1: first half-kick + drift + boundary (paper's F2), fused with the
// cell-count half of a2 (BIN): cell id and the slot handed out by the count atomic.
// ---------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ void boundary(T& r, T& v, T L, int bc, int* err)
{
    if (bc == BC_PERIODIC) {
        r = r - L * floor_(r / L);
        if (r >= L) r = r - L;
    } else if (bc == BC_REFLECT) {
        if (r < T(0)) { r = -r; v = -v; }
        else if (r > L) { r = T(2) * L - r; v = -v; }
        if (r < T(0) || r > L) *err = 1;
    }
}

// Geometric pore walls (the paper's own pore): one specular bounce per closed face whose
// rectangle the straight path r(t) -> r(t + dt) crosses, faces visited in the order -x, +x, -y, +y, -z, +z.
template <typename T>
__device__ __forceinline__ void prism_reflect(const Params<T>& p, const T (&ro)[3], T (&rn)[3], T (&vh)[3])
{
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int sgn = -1; sgn <= 1; sgn += 2) {
            if (a == p.prism_axis && sgn == 1) continue;                 // the open face
            const T w = p.prism_c[a] + T(sgn) * p.prism_h[a];
            if ((ro[a] - w) * (rn[a] - w) < T(0)) {
                const T t = (w - ro[a]) / (rn[a] - ro[a]);
                bool inside = true;
#pragma unroll
                for (int b = 0; b < 3; ++b)
                    if (b != a && fabs(ro[b] + t * (rn[b] - ro[b]) - p.prism_c[b]) > p.prism_h[b]) inside = false;
                if (inside) { rn[a] = T(2) * w - rn[a]; vh[a] = -vh[a]; }
            }
        }
}

template <typename T, bool MOVE, bool BIN>
__global__ void __launch_bounds__(256) k_kick_drift_bin(Params<T> p, State<T> s, Force<T> f, int* __restrict__ count,
                                                        int* __restrict__ cell, int* __restrict__ slot,
                                                        int* __restrict__ err)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.nv) return;
    Vec4<T> ri = s.r[i];
    T x = ri.x, y = ri.y, z = ri.z;
    if (MOVE) {
        T vx = s.vx[i] + p.hk * f.fx[i];
        T vy = s.vy[i] + p.hk * f.fy[i];
        T vz = s.vz[i] + p.hk * f.fz[i];
        x = x + p.dt * vx;
        y = y + p.dt * vy;
        z = z + p.dt * vz;
        if (p.prism) {
            const T ro[3] = {ri.x, ri.y, ri.z};
            T rn[3] = {x, y, z}, vh[3] = {vx, vy, vz};
            prism_reflect(p, ro, rn, vh);
            x = rn[0]; y = rn[1]; z = rn[2]; vx = vh[0]; vy = vh[1]; vz = vh[2];
        }
        boundary(x, vx, p.L[0], p.bc[0], err);
        boundary(y, vy, p.L[1], p.bc[1], err);
        boundary(z, vz, p.L[2], p.bc[2], err);
        ri.x = x; ri.y = y; ri.z = z;
        s.r[i] = ri;
        s.vx[i] = vx; s.vy[i] = vy; s.vz[i] = vz;
    }
    if (BIN) {
        int cx, cy, cz;
        int c = cell_index(p, x, y, z, cx, cy, cz);
        cell[i] = c;
        slot[i] = atomicAdd(&count[c], 1);
    }
}

// ---------------------------------------------------------------------------
// a2: exclusive prefix scan of the cell counts (two launches, no inter-block wait):
// k_scan_reduce sums tiles of SCAN_TILE counts; k_scan_apply adds the tile offsets,
// scans inside the tile with warp shuffles and zeroes the counts for the next step.
// ---------------------------------------------------------------------------
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

__device__ __forceinline__ int warp_incl_scan(int v)
{
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, v, d);
        if ((threadIdx.x & 31) >= d) v += t;
    }
    return v;
}

__device__ __forceinline__ int warp_sum(int v)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_reduce(const int* __restrict__ count, int n,
                                                              int* __restrict__ tile_sum)
{
    __shared__ int ws[SCAN_THREADS / 32];
    int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    int s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k)
        if (base + k < n) s += count[base + k];
    s = warp_sum(s);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        int t = threadIdx.x < SCAN_THREADS / 32 ? ws[threadIdx.x] : 0;
        t = warp_sum(t);
        if (threadIdx.x == 0) tile_sum[blockIdx.x] = t;
    }
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_apply(int* __restrict__ count, int n,
                                                             const int* __restrict__ tile_sum,
                                                             int* __restrict__ start)
{
    __shared__ int ws[SCAN_THREADS / 32];
    __shared__ int s_off;
    // offset of this tile = sum of the tile sums before it
    int off = 0;
    for (int k = threadIdx.x; k < (int)blockIdx.x; k += SCAN_THREADS) off += tile_sum[k];
    off = warp_sum(off);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = off;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
        for (int k = 0; k < SCAN_THREADS / 32; ++k) t += ws[k];
        s_off = t;
    }
    __syncthreads();
    off = s_off;
    __syncthreads();
    int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    int v[SCAN_ITEMS];
    int s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        v[k] = base + k < n ? count[base + k] : 0;
        s += v[k];
    }
    int incl = warp_incl_scan(s);
    if ((threadIdx.x & 31) == 31) ws[threadIdx.x >> 5] = incl;
    __syncthreads();
    int wofs = 0;
    for (int k = 0; k < (int)(threadIdx.x >> 5); ++k) wofs += ws[k];
    int run = off + wofs + incl - s;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (base + k < n) {
            start[base + k] = run;
            count[base + k] = 0;
        }
        run += v[k];
    }
    if (base <= n - 1 && n - 1 < base + SCAN_ITEMS) start[n] = run;
}

// a2: scatter of the particle state into cell order (ping-pong buffers).
template <typename T>
__global__ void __launch_bounds__(256) k_scatter(int nv, State<T> src, State<T> dst, Force<T> fsrc, Force<T> fdst,
                                                 const int* __restrict__ cell, const int* __restrict__ slot,
                                                 const int* __restrict__ start, int with_force)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nv) return;
    int d = start[cell[i]] + slot[i];
    dst.r[d] = src.r[i];
    dst.vx[d] = src.vx[i]; dst.vy[d] = src.vy[i]; dst.vz[d] = src.vz[i];
    dst.id[d] = src.id[i];
    if (with_force) { fdst.fx[d] = fsrc.fx[i]; fdst.fy[d] = fsrc.fy[i]; fdst.fz[d] = fsrc.fz[i]; }
}

// ---------------------------------------------------------------------------
// a3: pair term.  s = sigma^2 / r^2;  g = 24 eps (2 s^6 - s^3) / r^2;  u = 4 eps (s^6 - s^3) - u_c.
// Strict r^2 < r_c^2 with r^2 = fma(dz, dz, fma(dy, dy, dx*dx)) (reading A2).
// ---------------------------------------------------------------------------
template <typename T, bool ENERGY>
struct Acc {
    T fx = T(0), fy = T(0), fz = T(0);
    double u = 0.0, w = 0.0;
    int c = 0;
    long long tests = 0;
};

template <typename T, bool ENERGY>
__device__ __forceinline__ void pair_term(T dx, T dy, T dz, T rc2, T sig2, T e24, T e4, T uc, Acc<T, ENERGY>& a)
{
    T r2 = fma_(dz, dz, fma_(dy, dy, dx * dx));
    if (r2 < rc2) {
        T inv = T(1) / r2;
        T s = sig2 * inv;
        T s3 = s * s * s;
        T s6 = s3 * s3;
        T g = e24 * inv * (T(2) * s6 - s3);
        a.fx = fma_(g, dx, a.fx);
        a.fy = fma_(g, dy, a.fy);
        a.fz = fma_(g, dz, a.fz);
        if (ENERGY) {
            a.u += (double)(e4 * (s6 - s3) - uc);
            a.w += (double)(g * r2);
            a.c += 1;
        }
    }
}

// Variant B: cell-list traversal.  ROWS = 3^(d-1) lanes cooperate on one particle: lane `row` walks the
// cell row (cy+ky, cz+kz), whose three cells (cx-1, cx, cx+1) are contiguous in cell order, so a row is
// ONE contiguous j range (plus one wrapped cell at a periodic x face).  Images are applied by shifting
// r_i once per row/segment instead of a per-pair rint.  The ROWS partial sums are combined with warp
// shuffles in a fixed tree and the leader lane stores f_i and applies the second half-kick (a4).
// A warp holds 32 / ROWS particles (3 in 3D, 10 in 2D); short dependent chains and 9x the warps of a
// thread-per-particle walk are what hide the L2 latency at N ~ 1e5 (profiles/r01_v1_cfg2.md).
template <typename T, bool ENERGY>
__device__ __forceinline__ void row_range(const Vec4<T>* __restrict__ r, int jb, int je, int skip, T xe, T ye, T ze,
                                          T xj0, T yjs, T zjs, T rc2, T sig2, T e24, T e4, T uc, Acc<T, ENERGY>& a)
{
    constexpr bool TWO_SIDED = sizeof(T) == 4;
    for (int j = jb; j < je; j += 2) {
        const int j1 = min(j + 1, je - 1);
        const Vec4<T> a0 = r[j], a1 = r[j1];           // two independent loads in flight
        if (j != skip) {
            if (TWO_SIDED) pair_term<T, ENERGY>(xe - (a0.x - xj0), ye - (a0.y - yjs), ze - (a0.z - zjs), rc2, sig2, e24, e4, uc, a);
            else pair_term<T, ENERGY>(xe - a0.x, ye - a0.y, ze - a0.z, rc2, sig2, e24, e4, uc, a);
        }
        if (j1 != j && j1 != skip) {
            if (TWO_SIDED) pair_term<T, ENERGY>(xe - (a1.x - xj0), ye - (a1.y - yjs), ze - (a1.z - zjs), rc2, sig2, e24, e4, uc, a);
            else pair_term<T, ENERGY>(xe - a1.x, ye - a1.y, ze - a1.z, rc2, sig2, e24, e4, uc, a);
        }
    }
}

template <int ROWS, typename V>
__device__ __forceinline__ V rows_sum(V v, int row)
{
    constexpr int TOP = ROWS > 4 ? 8 : 2;    // largest power of two below ROWS (9 -> 8, 3 -> 2)
#pragma unroll
    for (int off = TOP; off > 0; off >>= 1) {
        V o = __shfl_down_sync(0xffffffffu, v, off);
        if (row < off && row + off < ROWS) v += o;
    }
    return v;
}

template <typename T, int ROWS, bool ENERGY, bool KICK, bool COUNT>
__global__ void __launch_bounds__(128) k_force_cells(Params<T> p, State<T> s, const int* __restrict__ start,
                                                     Walls<T> w, Force<T> f, EnergyOut eo,
                                                     unsigned long long* __restrict__ tests)
{
    constexpr int PPW = 32 / ROWS;
    constexpr bool TWO_SIDED = sizeof(T) == 4;
    const int lane = threadIdx.x & 31;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int pl = lane / ROWS, row = lane - pl * ROWS;
    const int i = warp * PPW + pl;
    const bool active = pl < PPW && i < p.nv;
    Acc<T, ENERGY> av, aw;
    long long nt = 0;
    if (active) {
        const Vec4<T> ri = s.r[i];
        int cx, cy, cz;
        const int ci = cell_index(p, ri.x, ri.y, ri.z, cx, cy, cz);
        const int nx = p.nc[0], ny = p.nc[1], nz = p.nc[2];
        const int ky = row % 3 - 1, kz = ROWS == 9 ? row / 3 - 1 : 0;
        int qy = cy + ky, qz = cz + kz;
        T ye = ri.y, ze = ri.z, yjs = T(0), zjs = T(0);
        bool ok = true;
        // image shifts: fp64 shifts r_i by +-L; fp32 puts the shift on whichever side sits at the top of
        // the box (r - L is exact there) so that d keeps full relative precision
        if (qz < 0) { ok = p.bc[2] == BC_PERIODIC; qz += nz; if (TWO_SIDED) zjs = p.L[2]; else ze += p.L[2]; }
        else if (qz >= nz) { ok = p.bc[2] == BC_PERIODIC; qz -= nz; ze -= p.L[2]; }
        if (qy < 0) { ok = ok && p.bc[1] == BC_PERIODIC; qy += ny; if (TWO_SIDED) yjs = p.L[1]; else ye += p.L[1]; }
        else if (qy >= ny) { ok = ok && p.bc[1] == BC_PERIODIC; qy -= ny; ye -= p.L[1]; }
        if (ok) {
            const int rowc = (qz * ny + qy) * nx;
            const int x0 = max(cx - 1, 0), x1 = min(cx + 1, nx - 1);
            int xw = -1;
            T xs = T(0), xjs = T(0);
            if (p.bc[0] == BC_PERIODIC) {
                if (cx == 0) { xw = nx - 1; if (TWO_SIDED) xjs = p.L[0]; else xs = p.L[0]; }
                else if (cx == nx - 1) { xw = 0; xs = -p.L[0]; }
            }
            const bool do_wall = p.nw > 0 && w.near[ci];
            // all cell-start loads first (independent), then the particle loops
            const int jb = start[rowc + x0], je = start[rowc + x1 + 1];
            int jb2 = 0, je2 = 0, wb = 0, we = 0, wb2 = 0, we2 = 0;
            if (xw >= 0) { jb2 = start[rowc + xw]; je2 = start[rowc + xw + 1]; }
            if (do_wall) {
                wb = w.start[rowc + x0]; we = w.start[rowc + x1 + 1];
                if (xw >= 0) { wb2 = w.start[rowc + xw]; we2 = w.start[rowc + xw + 1]; }
            }
            row_range<T, ENERGY>(s.r, jb, je, i, ri.x, ye, ze, T(0), yjs, zjs, p.rc2, p.sig2_vv, p.e24_vv, p.e4_vv,
                                 p.uc_vv, av);
            row_range<T, ENERGY>(s.r, jb2, je2, i, ri.x + xs, ye, ze, xjs, yjs, zjs, p.rc2, p.sig2_vv, p.e24_vv,
                                 p.e4_vv, p.uc_vv, av);
            row_range<T, ENERGY>(w.r, wb, we, -1, ri.x, ye, ze, T(0), yjs, zjs, p.rc2, p.sig2_vw, p.e24_vw, p.e4_vw,
                                 p.uc_vw, aw);
            row_range<T, ENERGY>(w.r, wb2, we2, -1, ri.x + xs, ye, ze, xjs, yjs, zjs, p.rc2, p.sig2_vw, p.e24_vw,
                                 p.e4_vw, p.uc_vw, aw);
            if (COUNT) {
                nt = (je - jb) + (je2 - jb2) + (we - wb) + (we2 - wb2);
                if ((i >= jb && i < je) || (i >= jb2 && i < je2)) nt -= 1;
            }
        }
    }
    const T fx = rows_sum<ROWS>(av.fx + aw.fx, row);
    const T fy = rows_sum<ROWS>(av.fy + aw.fy, row);
    const T fz = rows_sum<ROWS>(av.fz + aw.fz, row);
    double uv = 0, uw = 0, wv = 0, ww = 0;
    int cv = 0, cw = 0;
    if (ENERGY) {
        uv = rows_sum<ROWS>(av.u, row); uw = rows_sum<ROWS>(aw.u, row);
        wv = rows_sum<ROWS>(av.w, row); ww = rows_sum<ROWS>(aw.w, row);
        cv = rows_sum<ROWS>(av.c, row); cw = rows_sum<ROWS>(aw.c, row);
    }
    if (COUNT) nt = rows_sum<ROWS>(nt, row);
    if (!active || row != 0) return;
    f.fx[i] = fx; f.fy[i] = fy; f.fz[i] = fz;
    if (KICK) {   // a4: second half-kick (paper's F3)
        s.vx[i] = s.vx[i] + p.hk * fx;
        s.vy[i] = s.vy[i] + p.hk * fy;
        s.vz[i] = s.vz[i] + p.hk * fz;
    }
    if (ENERGY) {
        eo.pe[i] = 0.5 * uv + uw;
        eo.pew[i] = uw;
        eo.vir[i] = 0.5 * wv + ww;
        eo.cvv[i] = cv;
        eo.cvw[i] = cw;
    }
    if (COUNT) atomicAdd(tests, (unsigned long long)nt);
}

// Minimum image d - L rint(d / L).  fp64: fma(-L, rint(d * invL), d).  fp32: the image shift is applied to
// whichever particle sits at the top of the box (exact), then the difference is taken (exact for near pairs).
__device__ __forceinline__ double min_image(double, double, double d, double L, double invL)
{
    return fma(-L, rint(d * invL), d);
}
__device__ __forceinline__ float min_image(float a, float b, float d, float L, float invL)
{
    float n = rintf(d * invL);
    return (a - fmaxf(n, 0.f) * L) - (b + fminf(n, 0.f) * L);
}

// Variant A: all-pairs, j staged through shared-memory tiles, minimum image per pair
// (d <- d - L rint(d / L) as fma(-L, rint(d * invL), d)).  One thread per particle i.
constexpr int AP_THREADS = 128;

template <typename T, bool ENERGY, bool KICK>
__global__ void __launch_bounds__(AP_THREADS) k_force_allpairs(Params<T> p, State<T> s,
                                                               const Vec4<T>* __restrict__ wr, Force<T> f,
                                                               EnergyOut eo)
{
    __shared__ T sx[AP_THREADS], sy[AP_THREADS], sz[AP_THREADS];
    const int i = blockIdx.x * AP_THREADS + threadIdx.x;
    const bool live = i < p.nv;
    Vec4<T> ri = {T(0), T(0), T(0), T(0)};
    if (live) ri = s.r[i];
    const T xi = ri.x, yi = ri.y, zi = ri.z;
    const bool px = p.bc[0] == BC_PERIODIC, py = p.bc[1] == BC_PERIODIC, pz = p.bc[2] == BC_PERIODIC;
    Acc<T, ENERGY> av, aw;
    for (int pass = 0; pass < 2; ++pass) {
        const int n = pass == 0 ? p.nv : p.nw;
        const Vec4<T>* jr = pass == 0 ? s.r : wr;
        for (int t0 = 0; t0 < n; t0 += AP_THREADS) {
            int j = t0 + threadIdx.x;
            __syncthreads();
            if (j < n) { Vec4<T> q = jr[j]; sx[threadIdx.x] = q.x; sy[threadIdx.x] = q.y; sz[threadIdx.x] = q.z; }
            __syncthreads();
            const int m = min(AP_THREADS, n - t0);
#pragma unroll 4
            for (int k = 0; k < m; ++k) {
                if (pass == 0 && t0 + k == i) continue;
                T dx = xi - sx[k], dy = yi - sy[k], dz = zi - sz[k];
                if (px) dx = min_image(xi, sx[k], dx, p.L[0], p.invL[0]);
                if (py) dy = min_image(yi, sy[k], dy, p.L[1], p.invL[1]);
                if (pz) dz = min_image(zi, sz[k], dz, p.L[2], p.invL[2]);
                if (pass == 0)
                    pair_term<T, ENERGY>(dx, dy, dz, p.rc2, p.sig2_vv, p.e24_vv, p.e4_vv, p.uc_vv, av);
                else
                    pair_term<T, ENERGY>(dx, dy, dz, p.rc2, p.sig2_vw, p.e24_vw, p.e4_vw, p.uc_vw, aw);
            }
        }
    }
    if (!live) return;
    const T fx = av.fx + aw.fx, fy = av.fy + aw.fy, fz = av.fz + aw.fz;
    f.fx[i] = fx; f.fy[i] = fy; f.fz[i] = fz;
    if (KICK) {
        s.vx[i] = s.vx[i] + p.hk * fx;
        s.vy[i] = s.vy[i] + p.hk * fy;
        s.vz[i] = s.vz[i] + p.hk * fz;
    }
    if (ENERGY) {
        eo.pe[i] = 0.5 * av.u + aw.u;
        eo.pew[i] = aw.u;
        eo.vir[i] = 0.5 * av.w + aw.w;
        eo.cvv[i] = av.c;
        eo.cvw[i] = aw.c;
    }
}

// ---------------------------------------------------------------------------
// boundary helpers: AoS fp64 [n][dim] (caller's order) <-> SoA T (internal order)
// ---------------------------------------------------------------------------
template <typename T>
__global__ void k_import(int n, int dim, const double* __restrict__ pos, const double* __restrict__ vel, State<T> s)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    Vec4<T> r;
    r.x = (T)pos[i * dim];
    r.y = (T)pos[i * dim + 1];
    r.z = dim == 3 ? (T)pos[i * dim + 2] : T(0);
    r.w = T(0);
    s.r[i] = r;
    if (vel) {
        s.vx[i] = (T)vel[i * dim];
        s.vy[i] = (T)vel[i * dim + 1];
        s.vz[i] = dim == 3 ? (T)vel[i * dim + 2] : T(0);
    }
    if (s.id) s.id[i] = i;
}

// out[id[i]][0..dim) = (a[i], b[i], c[i])
template <typename T>
__global__ void k_export3(int n, int dim, const int* __restrict__ id, const T* __restrict__ a, const T* __restrict__ b,
                          const T* __restrict__ c, double* __restrict__ out)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    size_t o = (size_t)id[i] * dim;
    out[o] = (double)a[i];
    out[o + 1] = (double)b[i];
    if (dim == 3) out[o + 2] = (double)c[i];
}

__global__ void k_export1(int n, const int* __restrict__ id, const double* __restrict__ a, double* __restrict__ out)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[id[i]] = a[i];
}

// out[id[i]][0..dim) = r[i].xyz
template <typename T>
__global__ void k_export_pos(int n, int dim, const int* __restrict__ id, const Vec4<T>* __restrict__ r,
                             double* __restrict__ out)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    size_t o = (size_t)id[i] * dim;
    Vec4<T> v = r[i];
    out[o] = (double)v.x;
    out[o + 1] = (double)v.y;
    if (dim == 3) out[o + 2] = (double)v.z;
}

// near[c] = 1 if any of the 3^d neighbour cells of c (same wrap / drop rule as the force
// kernel) holds a wall particle.  Run once at create (walls never move).
template <typename T>
__global__ void k_wall_near(Params<T> p, const int* __restrict__ wstart, uint8_t* __restrict__ near)
{
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= p.ncell) return;
    int cx = c % p.nc[0], cy = (c / p.nc[0]) % p.nc[1], cz = c / (p.nc[0] * p.nc[1]);
    int any = 0;
    for (int kz = -1; kz <= 1; ++kz)
        for (int ky = -1; ky <= 1; ++ky)
            for (int kx = -1; kx <= 1; ++kx) {
                int q[3] = {cx + kx, cy + ky, cz + kz};
                bool ok = true;
                for (int a = 0; a < 3; ++a) {
                    if (q[a] < 0 || q[a] >= p.nc[a]) {
                        if (p.bc[a] == BC_PERIODIC) q[a] = (q[a] + p.nc[a]) % p.nc[a];
                        else ok = false;
                    }
                }
                if (!ok) continue;
                int cj = (q[2] * p.nc[1] + q[1]) * p.nc[0] + q[0];
                any |= (wstart[cj + 1] - wstart[cj]) > 0;
            }
    near[c] = (uint8_t)any;
}

// ---------------------------------------------------------------------------
// a5: energy reductions.  Warp shuffle -> block -> per-block partials; a second
// single-block launch sums the partials in a fixed order (deterministic for a given
// particle order).  part layout: [6][nblocks]: K, U, U_vw, virial, ordered vv hits, vw hits.
// ---------------------------------------------------------------------------
constexpr int RED_THREADS = 256;

__device__ __forceinline__ double warp_sum_d(double v)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

__device__ __forceinline__ void block_sum6(double (&v)[6], double* out, int stride)
{
    __shared__ double sh[6][RED_THREADS / 32];
#pragma unroll
    for (int q = 0; q < 6; ++q) {
        double t = warp_sum_d(v[q]);
        if ((threadIdx.x & 31) == 0) sh[q][threadIdx.x >> 5] = t;
    }
    __syncthreads();
    if (threadIdx.x < 6) {
        double t = 0.0;
        for (int k = 0; k < RED_THREADS / 32; ++k) t += sh[threadIdx.x][k];
        out[threadIdx.x * stride] = t;
    }
}

template <typename T>
__global__ void __launch_bounds__(RED_THREADS) k_energy_partial(int n, double mass, State<T> s, EnergyOut eo,
                                                                double* __restrict__ part)
{
    double v[6] = {0, 0, 0, 0, 0, 0};
    for (int i = blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += gridDim.x * RED_THREADS) {
        double vx = (double)s.vx[i], vy = (double)s.vy[i], vz = (double)s.vz[i];
        v[0] += 0.5 * mass * (vx * vx + vy * vy + vz * vz);
        v[1] += eo.pe[i];
        v[2] += eo.pew[i];
        v[3] += eo.vir[i];
        v[4] += (double)eo.cvv[i];
        v[5] += (double)eo.cvw[i];
    }
    block_sum6(v, part + blockIdx.x, gridDim.x);
}

__global__ void __launch_bounds__(RED_THREADS) k_energy_final(int nblocks, const double* __restrict__ part,
                                                              double* __restrict__ out)
{
    double v[6] = {0, 0, 0, 0, 0, 0};
    for (int b = threadIdx.x; b < nblocks; b += RED_THREADS)
#pragma unroll
        for (int q = 0; q < 6; ++q) v[q] += part[q * nblocks + b];
    block_sum6(v, out, 1);
}

// NEXT-2, virial pressure: per-block sums of K and W over all particles and over the particles
// inside the pore region; part layout [6][nblocks]: K_all, W_all, K_in, W_in, n_in, 0 (summed by k_energy_final).
struct PoreRegion {
    int kind;          // 0 none, 1 slit (2D), 2 cylinder (3D)
    int axis;
    double c[3], half_len, r0sq, half_width;
};

template <typename T>
__global__ void __launch_bounds__(RED_THREADS) k_pressure_partial(Params<T> p, State<T> s, const double* __restrict__ vir,
                                                                 PoreRegion g, double* __restrict__ part)
{
    double v[6] = {0, 0, 0, 0, 0, 0};
    for (int i = blockIdx.x * RED_THREADS + threadIdx.x; i < p.nv; i += gridDim.x * RED_THREADS) {
        const double vx = (double)s.vx[i], vy = (double)s.vy[i], vz = (double)s.vz[i];
        const double k = 0.5 * p.mass * (vx * vx + vy * vy + vz * vz), w = vir[i];
        Vec4<T> ri = s.r[i];
        T dummy = T(0);
        int err = 0;
        boundary(ri.x, dummy, p.L[0], p.bc[0] == BC_PERIODIC ? BC_PERIODIC : BC_NONE, &err);   // VERLET keeps them unwrapped
        boundary(ri.y, dummy, p.L[1], p.bc[1] == BC_PERIODIC ? BC_PERIODIC : BC_NONE, &err);
        boundary(ri.z, dummy, p.L[2], p.bc[2] == BC_PERIODIC ? BC_PERIODIC : BC_NONE, &err);
        const double d[3] = {(double)ri.x - g.c[0], (double)ri.y - g.c[1], (double)ri.z - g.c[2]};
        bool in = false;
        if (g.kind == 1) in = fabs(d[g.axis]) < g.half_width && fabs(d[1 - g.axis]) < g.half_len;
        else if (g.kind == 2) {
            const int a1 = (g.axis + 1) % 3, a2 = (g.axis + 2) % 3;
            in = fabs(d[g.axis]) < g.half_len && d[a1] * d[a1] + d[a2] * d[a2] < g.r0sq;
        }
        v[0] += k; v[1] += w;
        if (in) { v[2] += k; v[3] += w; v[4] += 1.0; }
    }
    block_sum6(v, part + blockIdx.x, gridDim.x);
}

// NEXT-4: density profiles about the pore, integer histograms (shared-memory bins, then global atomics).
constexpr int HIST_MAX_BINS = 1024;

template <typename T>
__global__ void __launch_bounds__(256) k_density_profile(Params<T> p, State<T> s, PoreRegion g, int along_dim, double box_len,
                                                         int n_axial, int n_radial, double r_max,
                                                         unsigned long long* __restrict__ out)
{
    __shared__ unsigned int bins[HIST_MAX_BINS];
    const int nb = n_axial + n_radial;
    for (int k = threadIdx.x; k < nb; k += blockDim.x) bins[k] = 0;
    __syncthreads();
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < p.nv; i += gridDim.x * blockDim.x) {
        Vec4<T> ri = s.r[i];
        T dummy = T(0);
        int err = 0;
        boundary(ri.x, dummy, p.L[0], p.bc[0] == BC_PERIODIC ? BC_PERIODIC : BC_NONE, &err);
        boundary(ri.y, dummy, p.L[1], p.bc[1] == BC_PERIODIC ? BC_PERIODIC : BC_NONE, &err);
        boundary(ri.z, dummy, p.L[2], p.bc[2] == BC_PERIODIC ? BC_PERIODIC : BC_NONE, &err);
        const double x[3] = {(double)ri.x, (double)ri.y, (double)ri.z};
        if (n_axial > 0) {
            const int b = min(max((int)floor(x[along_dim] / box_len * n_axial), 0), n_axial - 1);
            atomicAdd(&bins[b], 1u);
        }
        if (n_radial > 0) {
            const double d[3] = {x[0] - g.c[0], x[1] - g.c[1], x[2] - g.c[2]};
            double rho;
            bool in;
            if (g.kind == 1) { rho = fabs(d[g.axis]); in = fabs(d[1 - g.axis]) < g.half_len; }
            else {
                const int a1 = (g.axis + 1) % 3, a2 = (g.axis + 2) % 3;
                rho = sqrt(d[a1] * d[a1] + d[a2] * d[a2]); in = fabs(d[g.axis]) < g.half_len;
            }
            const int b = (int)floor(rho / r_max * n_radial);
            if (in && b >= 0 && b < n_radial) atomicAdd(&bins[n_axial + b], 1u);
        }
    }
    __syncthreads();
    for (int k = threadIdx.x; k < nb; k += blockDim.x)
        if (bins[k]) atomicAdd(&out[k], (unsigned long long)bins[k]);
}

// ---------------------------------------------------------------------------
// F4, Berendsen thermostat for the multi-kernel paths: block partial sums of K, then every
// block re-sums the partials in the same fixed order, forms lambda and rescales its velocities.
// ---------------------------------------------------------------------------
__device__ __forceinline__ double berendsen_lambda(double kinetic, double rate, double t_target, double dof)
{
    const double T = 2.0 * kinetic / dof;
    return T > 0.0 ? sqrt(1.0 + rate * (t_target / T - 1.0)) : 1.0;
}

template <typename T>
__global__ void __launch_bounds__(RED_THREADS) k_kinetic_partial(int n, double mass, State<T> s, double* __restrict__ part)
{
    __shared__ double sh[RED_THREADS / 32];
    double k = 0.0;
    for (int i = blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += gridDim.x * RED_THREADS) {
        const double vx = (double)s.vx[i], vy = (double)s.vy[i], vz = (double)s.vz[i];
        k += 0.5 * mass * (vx * vx + vy * vy + vz * vz);
    }
    k = warp_sum_d(k);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = k;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int q = 0; q < RED_THREADS / 32; ++q) t += sh[q];
        part[blockIdx.x] = t;
    }
}

template <typename T>
__global__ void __launch_bounds__(256) k_thermo_scale(Params<T> p, State<T> s, int nblocks, const double* __restrict__ part)
{
    __shared__ double s_lambda;
    if (threadIdx.x == 0) {
        double k = 0.0;
        for (int b = 0; b < nblocks; ++b) k += part[b];
        s_lambda = berendsen_lambda(k, p.thermo_rate, p.t_target, p.dof);
    }
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.nv) return;
    const T lam = (T)s_lambda;
    s.vx[i] = lam * s.vx[i]; s.vy[i] = lam * s.vy[i]; s.vz[i] = lam * s.vz[i];
}

// ---------------------------------------------------------------------------
// peak micro-benchmarks (roofline denominators measured in the same run)
// ---------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) k_fma_chain(int iters, T seed, T* __restrict__ out)
{
    T a[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) a[k] = seed + T(k) + T(threadIdx.x) * T(1e-3);
    const T m = T(0.999999), c = T(1e-7);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) a[k] = fma_(a[k], m, c);
    }
    T sum = T(0);
#pragma unroll
    for (int k = 0; k < 8; ++k) sum += a[k];
    if (sum == T(-1)) out[blockIdx.x * blockDim.x + threadIdx.x] = sum;
}

__global__ void __launch_bounds__(256) k_copy(const double2* __restrict__ a, double2* __restrict__ b, size_t n)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        b[i] = a[i];
}

} // namespace md
