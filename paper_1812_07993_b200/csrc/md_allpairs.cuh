// md_allpairs.cuh -- variant A of a3 for fp64: all-pairs force kernel bound by the FP64 pipe.
//
// The paper's F1 tests every pair (Fig. 1 at :69-73).  With r_c = 2.5 sigma only ~5e-5 of
// the tests at N = 65,536 are hits, so the kernel is the distance TEST, and the test is written to cost
// three FP64 instructions:
//     t = |r_i|^2 - r^2 = 2 x_i x_j + 2 y_i y_j + 2 z_i z_j - |r_j|^2      3 DFMA  (6 flops)
//     r^2 < r_c^2  <=>  t > |r_i|^2 - r_c^2                                  (a threshold per particle i)
// with (x_j, y_j, z_j, -|r_j|^2) staged through shared memory as one 32-byte entry (its last word starts the chain),
// four particles i per thread in registers, and the comparison done by the integer pipe: the origin of the
// coordinates is placed so that |r_i|^2 > r_c^2 + margin for every particle i (x is measured from r_c + 1 sigma
// outside the box), hence every threshold is a positive double, positive doubles order like their high words, and a
// negative t (a pair further apart than |r_i|) is a negative integer.  One running integer maximum per particle i
// replaces the compare.  The form loses ~1e-11 absolute, and the high word of a value near |r_i|^2 has a grain of up
// to 2^-20 |r_i|^2, so it is only a conservative FILTER: a group of tests with any candidate re-evaluates its pairs
// exactly -- d = r_i - r_j, r^2 = fma(dz,dz,fma(dy,dy,dx*dx)), strict r^2 < r_c^2 -- and only that exact path
// produces forces and energies.  (Until the last hours of round 2 the filter value was r^2 itself: 1 DADD + 3 DFMA.)
// Periodic images are materialised once per step as ghost entries (particles within r_c of a periodic
// face), so the inner loop has no minimum-image arithmetic.  y and z are centred on the box middle to keep |r|^2
// small.  The fp32 variant is at the end of this file; boxes with a periodic length below 2.2 r_c
// (more than one image per dimension) keep the per-pair minimum-image kernel of md_kernels.cuh.
#pragma once
#include "md_kernels.cuh"

namespace md {

constexpr int AD_THREADS = 128;   // threads per block = entries per shared-memory tile
#ifndef MD_AD_IB
#define MD_AD_IB 4
#endif
#ifndef MD_AD_UNROLL
#define MD_AD_UNROLL 16
#endif
constexpr int AD_IB = MD_AD_IB;   // particles i per thread for large N; 1 below AD_SMALL_N (more, shorter blocks: the
constexpr int AD_SMALL_N = 8192;  // kernel is latency-bound there, profiles/r01_final_cfg2.md)
constexpr int AD_UNROLL = MD_AD_UNROLL;   // tests per i between two candidate checks
#ifndef MD_AD_JB
#define MD_AD_JB 4
#endif
constexpr int AD_JB = MD_AD_JB;           // list entries whose tests are advanced together, stage by stage

struct AllPairsDot {
    Vec4<double>* jv;      // [nv + cap_ghost]: real vapor entries in particle order, then this step's ghosts
    Vec4<double>* jw;      // [nwg]: wall particles and their ghosts (static)
    int* ghost_count;      // number of vapor ghosts appended this step
    int nwg;
    double thr;            // r_c^2 + rounding bound: candidate iff hi32(t) >= hi32(|r_i|^2 - thr)
    double org[3];         // origin of the stored coordinates (entry = r - org): x: -(r_c + 1), y and z: box centre
    double edge;           // r_c + margin: distance from a periodic face that spawns a ghost
};

// Appends (x, y, z) -- already centred -- and its periodic images to a j list.
__device__ __forceinline__ void push_images(const Params<double>& p, const AllPairsDot& a, double x, double y, double z,
                                            Vec4<double>* __restrict__ out, int base, int* __restrict__ counter)
{
    // shift options per dimension: 0, and +-L when within `edge` of the opposite face
    double sx[2] = {0.0, 0.0}, sy[2] = {0.0, 0.0}, sz[2] = {0.0, 0.0};
    int nx = 1, ny = 1, nz = 1;
    // the box is [-org, L - org) in the stored coordinates
    if (p.bc[0] == BC_PERIODIC) { if (x < a.edge - a.org[0]) sx[nx++] = p.L[0]; else if (x > p.L[0] - a.org[0] - a.edge) sx[nx++] = -p.L[0]; }
    if (p.bc[1] == BC_PERIODIC) { if (y < a.edge - a.org[1]) sy[ny++] = p.L[1]; else if (y > p.L[1] - a.org[1] - a.edge) sy[ny++] = -p.L[1]; }
    if (p.bc[2] == BC_PERIODIC) { if (z < a.edge - a.org[2]) sz[nz++] = p.L[2]; else if (z > p.L[2] - a.org[2] - a.edge) sz[nz++] = -p.L[2]; }
    for (int c = 0; c < nz; ++c)
        for (int b = 0; b < ny; ++b)
            for (int q = 0; q < nx; ++q) {
                if (q + b + c == 0) continue;
                Vec4<double> e;
                e.x = x + sx[q]; e.y = y + sy[b]; e.z = z + sz[c];
                e.w = -fma(e.z, e.z, fma(e.y, e.y, e.x * e.x));
                out[base + atomicAdd(counter, 1)] = e;
            }
}

// a1 for the all-pairs path: half-kick + drift + boundary, then the step's j list (entry + ghosts); f is
// cleared for the force kernel's accumulation.  MOVE = false only builds the list (md_create).
template <bool MOVE>
__global__ void __launch_bounds__(256) k_ap_kick_drift_list(Params<double> p, State<double> s, Force<double> f,
                                                            AllPairsDot a, int* __restrict__ err)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.nv) return;
    Vec4<double> ri = s.r[i];
    if (MOVE) {
        double vx = s.vx[i] + p.hk * f.fx[i];
        double vy = s.vy[i] + p.hk * f.fy[i];
        double vz = s.vz[i] + p.hk * f.fz[i];
        {
            const double ro[3] = {ri.x, ri.y, ri.z};
            double rn[3] = {ri.x + p.dt * vx, ri.y + p.dt * vy, ri.z + p.dt * vz}, vh[3] = {vx, vy, vz};
            if (p.prism) prism_reflect(p, ro, rn, vh);
            ri.x = rn[0]; ri.y = rn[1]; ri.z = rn[2]; vx = vh[0]; vy = vh[1]; vz = vh[2];
        }
        boundary(ri.x, vx, p.L[0], p.bc[0], err);
        boundary(ri.y, vy, p.L[1], p.bc[1], err);
        boundary(ri.z, vz, p.L[2], p.bc[2], err);
        s.r[i] = ri;
        s.vx[i] = vx; s.vy[i] = vy; s.vz[i] = vz;
    }
    f.fx[i] = 0.0; f.fy[i] = 0.0; f.fz[i] = 0.0;
    Vec4<double> e;
    e.x = ri.x - a.org[0]; e.y = ri.y - a.org[1]; e.z = ri.z - a.org[2];
    e.w = -fma(e.z, e.z, fma(e.y, e.y, e.x * e.x));
    a.jv[i] = e;
    push_images(p, a, e.x, e.y, e.z, a.jv, p.nv, a.ghost_count);
}

// Static wall list (md_create): entry + ghosts of every wall particle.
__global__ void k_ap_wall_list(Params<double> p, const Vec4<double>* __restrict__ wr, AllPairsDot a, int* __restrict__ counter)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.nw) return;
    Vec4<double> e;
    e.x = wr[i].x - a.org[0]; e.y = wr[i].y - a.org[1]; e.z = wr[i].z - a.org[2];
    e.w = -fma(e.z, e.z, fma(e.y, e.y, e.x * e.x));
    a.jw[i] = e;
    push_images(p, a, e.x, e.y, e.z, a.jw, p.nw, counter);
}

// a4 for the all-pairs path: second half-kick once every block's force contributions have landed; also
// re-arms the ghost counter for the next step.
template <typename T>
__global__ void __launch_bounds__(256) k_ap_kick(Params<T> p, State<T> s, Force<T> f, int* __restrict__ ghost_count)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) *ghost_count = 0;
    if (i >= p.nv) return;
    s.vx[i] = s.vx[i] + p.hk * f.fx[i];
    s.vy[i] = s.vy[i] + p.hk * f.fy[i];
    s.vz[i] = s.vz[i] + p.hk * f.fz[i];
}

// Exact re-evaluation of one (i, j) pair found by the filter (reading A2: strict r^2 < r_c^2).
template <bool ENERGY>
__device__ __forceinline__ void ap_exact(const Params<double>& p, bool wall, double xi, double yi, double zi,
                                         const Vec4<double>& q, double& fx, double& fy, double& fz, double& u, double& w,
                                         int& c)
{
    const double dx = xi - q.x, dy = yi - q.y, dz = zi - q.z;
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    if (r2 < p.rc2) {
        const double inv = 1.0 / r2;
        const double s = (wall ? p.sig2_vw : p.sig2_vv) * inv;
        const double s3 = s * s * s, s6 = s3 * s3;
        const double g = (wall ? p.e24_vw : p.e24_vv) * inv * (2.0 * s6 - s3);
        fx = fma(g, dx, fx); fy = fma(g, dy, fy); fz = fma(g, dz, fz);
        if (ENERGY) {
            u += (wall ? p.e4_vw : p.e4_vv) * (s6 - s3) - (wall ? p.uc_vw : p.uc_vv);
            w += g * r2;
            c += 1;
        }
    }
}

// grid = (i blocks, j slices).  Block (bi, sj) owns particles [bi * 128 IB, (bi + 1) * 128 IB) (thread t: i = base +
// t + 128 b, b < IB) and the tiles t with t % gridDim.y == sj of the j lists (vapor + ghosts, then walls).
// Forces are accumulated with fp64 atomics (f was cleared by k_ap_kick_drift_list); ENERGY instead
// accumulates pe, pe_w, virial and hit counts (cleared by the host) and leaves f alone.
template <bool ENERGY, int IB>
__global__ void __launch_bounds__(AD_THREADS) k_force_allpairs_dot(Params<double> p, AllPairsDot a, Force<double> f,
                                                                   EnergyOut eo)
{
    __shared__ Vec4<double> sjb[2][AD_THREADS];            // two tiles: one barrier per tile (see the loop)
    const int base = blockIdx.x * (AD_THREADS * IB) + threadIdx.x;
    double ax[IB], ay[IB], az[IB];              // 2 x_i, 2 y_i, 2 z_i
    int idx[IB], thr[IB];                       // thr: high word of |r_i|^2 - (r_c^2 + rounding bound) > 0
#pragma unroll
    for (int b = 0; b < IB; ++b) {
        idx[b] = base + b * AD_THREADS;
        // particles beyond nv: parked far away so that they never pass the filter
        Vec4<double> e = {1.0e9, 1.0e9, 1.0e9, -3.0e18};
        if (idx[b] < p.nv) e = a.jv[idx[b]];
        ax[b] = 2.0 * e.x; ay[b] = 2.0 * e.y; az[b] = 2.0 * e.z;
        thr[b] = __double2hiint(-e.w - a.thr);
    }
    double fx[IB] = {}, fy[IB] = {}, fz[IB] = {}, uv[IB] = {}, uw[IB] = {}, wv[IB] = {}, ww[IB] = {};
    int cv[IB] = {}, cw[IB] = {};
    bool any = false;
    const int nvj = p.nv + *a.ghost_count;
    const int tiles_v = (nvj + AD_THREADS - 1) / AD_THREADS, tiles_w = (a.nwg + AD_THREADS - 1) / AD_THREADS;
    // the tile after the current one is fetched into a register while the current one is evaluated, so a block never
    // waits for a global load between two tiles (it did: two barriers and an L2 round trip every 128 entries)
    auto fetch = [&](int t) {
        Vec4<double> e = {-1.0e9, -1.0e9, -1.0e9, -3.0e18};             // padding: far from everything
        if (t < tiles_v + tiles_w) {
            const bool w = t >= tiles_v;
            const int j = (w ? t - tiles_v : t) * AD_THREADS + threadIdx.x;
            if (j < (w ? a.nwg : nvj)) e = (w ? a.jw : a.jv)[j];
        }
        return e;
    };
    // Tile t is evaluated from buffer `cur` while tile t + gridDim.y is written into the other one, whose previous
    // contents (the tile before t) every warp finished before it passed the barrier that published tile t.
    int cur = 0;
    sjb[0][threadIdx.x] = fetch(blockIdx.y);
    Vec4<double> nxt = fetch(blockIdx.y + gridDim.y);
    for (int t = blockIdx.y; t < tiles_v + tiles_w; t += gridDim.y, cur ^= 1) {
        const bool wall = t >= tiles_v;
        const int j0 = (wall ? t - tiles_v : t) * AD_THREADS;
        __syncthreads();
        sjb[cur ^ 1][threadIdx.x] = nxt;
        nxt = fetch(t + 2 * gridDim.y);
        const Vec4<double>* __restrict__ sj = sjb[cur];
        for (int k0 = 0; k0 < AD_THREADS; k0 += AD_UNROLL) {
            // one integer instruction per test beside the three FP64 ones: the running maximum, per particle i, of the
            // high words of t (t > 0 orders like its high word; t < 0 is a negative integer and never the maximum)
            int top[IB];
#pragma unroll
            for (int b = 0; b < IB; ++b) top[b] = (int)0x80000000;
#pragma unroll
            for (int u = 0; u < AD_UNROLL; u += AD_JB) {
                // AD_JB entries x IB particles independent chains, advanced one stage at a time
                Vec4<double> q[AD_JB];
                double t[AD_JB][IB];
#pragma unroll
                for (int w = 0; w < AD_JB; ++w) q[w] = sj[k0 + u + w];
#pragma unroll
                for (int w = 0; w < AD_JB; ++w)
#pragma unroll
                    for (int b = 0; b < IB; ++b) t[w][b] = fma(q[w].z, az[b], q[w].w);
#pragma unroll
                for (int w = 0; w < AD_JB; ++w)
#pragma unroll
                    for (int b = 0; b < IB; ++b) t[w][b] = fma(q[w].y, ay[b], t[w][b]);
#pragma unroll
                for (int w = 0; w < AD_JB; ++w)
#pragma unroll
                    for (int b = 0; b < IB; ++b) t[w][b] = fma(q[w].x, ax[b], t[w][b]);
#pragma unroll
                for (int w = 0; w < AD_JB; ++w)
#pragma unroll
                    for (int b = 0; b < IB; ++b) top[b] = max(top[b], __double2hiint(t[w][b]));
            }
            bool cand = false;
#pragma unroll
            for (int b = 0; b < IB; ++b) cand |= top[b] >= thr[b];
            if (cand) {              // this lane has a candidate in the group: it redoes ITS flagged pairs exactly
                for (int u = 0; u < AD_UNROLL; ++u) {
                    const Vec4<double> q = sj[k0 + u];
#pragma unroll
                    for (int b = 0; b < IB; ++b) {
                        const double t = fma(ax[b], q.x, fma(ay[b], q.y, fma(az[b], q.z, q.w)));
                        if (__double2hiint(t) < thr[b]) continue;              // same filter value as above
                        if (!wall && j0 + k0 + u == idx[b]) continue;          // j == i skipped by index
                        if (wall) ap_exact<ENERGY>(p, true, 0.5 * ax[b], 0.5 * ay[b], 0.5 * az[b], q, fx[b], fy[b], fz[b], uw[b], ww[b], cw[b]);
                        else ap_exact<ENERGY>(p, false, 0.5 * ax[b], 0.5 * ay[b], 0.5 * az[b], q, fx[b], fy[b], fz[b], uv[b], wv[b], cv[b]);
                    }
                }
                any = true;
            }
        }
    }
    if (!any) return;
#pragma unroll
    for (int b = 0; b < IB; ++b) {
        const int i = idx[b];
        if (i >= p.nv) continue;
        if (!ENERGY) {
            if (fx[b] != 0.0 || fy[b] != 0.0 || fz[b] != 0.0) {
                atomicAdd(&f.fx[i], fx[b]); atomicAdd(&f.fy[i], fy[b]); atomicAdd(&f.fz[i], fz[b]);
            }
        } else if (cv[b] | cw[b]) {
            atomicAdd(&eo.pe[i], 0.5 * uv[b] + uw[b]);
            atomicAdd(&eo.pew[i], uw[b]);
            atomicAdd(&eo.vir[i], 0.5 * wv[b] + ww[b]);
            atomicAdd(&eo.cvv[i], cv[b]);
            atomicAdd(&eo.cvw[i], cw[b]);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// fp32 mode of the same kernel.  The filter is the same three-instruction form in FP32 (3 FFMA, running integer
// maximum of the float's bits per particle i); its rounding (~1e-6 |r|^2) is covered by a wider margin.  Candidates
// are NOT re-evaluated from the shifted ghost entries -- a ghost coordinate x +- L rounded to fp32 would cost 4e-6
// sigma -- but from the original positions with the two-sided minimum image of md_kernels.cuh (exact differences
// for near pairs), found through the original index every entry carries.
// ---------------------------------------------------------------------------------------------------------
struct AllPairsDotF {
    Vec4<float>* jv;  int* jv_id;      // vapor entries + ghosts; id = particle index
    Vec4<float>* jw;  int* jw_id;      // wall entries + ghosts (static); id = wall index (caller order)
    const Vec4<float>* wr;             // wall positions, caller order
    int* ghost_count;
    int nwg;
    float thr;                         // r_c^2 + rounding bound: candidate iff bits(t) >= bits(|r_i|^2 - thr)
    float org[3];                      // origin of the stored coordinates, as AllPairsDot::org
    float edge;
};

__device__ __forceinline__ void push_images_f(const Params<float>& p, const AllPairsDotF& a, float x, float y, float z, int id,
                                              Vec4<float>* __restrict__ out, int* __restrict__ out_id, int base,
                                              int* __restrict__ counter)
{
    float sx[2] = {0.f, 0.f}, sy[2] = {0.f, 0.f}, sz[2] = {0.f, 0.f};
    int nx = 1, ny = 1, nz = 1;
    if (p.bc[0] == BC_PERIODIC) { if (x < a.edge - a.org[0]) sx[nx++] = p.L[0]; else if (x > p.L[0] - a.org[0] - a.edge) sx[nx++] = -p.L[0]; }
    if (p.bc[1] == BC_PERIODIC) { if (y < a.edge - a.org[1]) sy[ny++] = p.L[1]; else if (y > p.L[1] - a.org[1] - a.edge) sy[ny++] = -p.L[1]; }
    if (p.bc[2] == BC_PERIODIC) { if (z < a.edge - a.org[2]) sz[nz++] = p.L[2]; else if (z > p.L[2] - a.org[2] - a.edge) sz[nz++] = -p.L[2]; }
    for (int c = 0; c < nz; ++c)
        for (int b = 0; b < ny; ++b)
            for (int q = 0; q < nx; ++q) {
                if (q + b + c == 0) continue;
                Vec4<float> e;
                e.x = x + sx[q]; e.y = y + sy[b]; e.z = z + sz[c];
                e.w = -fmaf(e.z, e.z, fmaf(e.y, e.y, e.x * e.x));
                const int k = base + atomicAdd(counter, 1);
                out[k] = e;
                out_id[k] = id;
            }
}

template <bool MOVE>
__global__ void __launch_bounds__(256) k_apf_kick_drift_list(Params<float> p, State<float> s, Force<float> f,
                                                             AllPairsDotF a, int* __restrict__ err)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.nv) return;
    Vec4<float> ri = s.r[i];
    if (MOVE) {
        float vx = s.vx[i] + p.hk * f.fx[i];
        float vy = s.vy[i] + p.hk * f.fy[i];
        float vz = s.vz[i] + p.hk * f.fz[i];
        {
            const float ro[3] = {ri.x, ri.y, ri.z};
            float rn[3] = {ri.x + p.dt * vx, ri.y + p.dt * vy, ri.z + p.dt * vz}, vh[3] = {vx, vy, vz};
            if (p.prism) prism_reflect(p, ro, rn, vh);
            ri.x = rn[0]; ri.y = rn[1]; ri.z = rn[2]; vx = vh[0]; vy = vh[1]; vz = vh[2];
        }
        boundary(ri.x, vx, p.L[0], p.bc[0], err);
        boundary(ri.y, vy, p.L[1], p.bc[1], err);
        boundary(ri.z, vz, p.L[2], p.bc[2], err);
        s.r[i] = ri;
        s.vx[i] = vx; s.vy[i] = vy; s.vz[i] = vz;
    }
    f.fx[i] = 0.f; f.fy[i] = 0.f; f.fz[i] = 0.f;
    Vec4<float> e;
    e.x = ri.x - a.org[0]; e.y = ri.y - a.org[1]; e.z = ri.z - a.org[2];
    e.w = -fmaf(e.z, e.z, fmaf(e.y, e.y, e.x * e.x));
    a.jv[i] = e;
    a.jv_id[i] = i;
    push_images_f(p, a, e.x, e.y, e.z, i, a.jv, a.jv_id, p.nv, a.ghost_count);
}

__global__ void k_apf_wall_list(Params<float> p, AllPairsDotF a, int* __restrict__ counter)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.nw) return;
    Vec4<float> e;
    e.x = a.wr[i].x - a.org[0]; e.y = a.wr[i].y - a.org[1]; e.z = a.wr[i].z - a.org[2];
    e.w = -fmaf(e.z, e.z, fmaf(e.y, e.y, e.x * e.x));
    a.jw[i] = e;
    a.jw_id[i] = i;
    push_images_f(p, a, e.x, e.y, e.z, i, a.jw, a.jw_id, p.nw, counter);
}

template <bool ENERGY, int IB>
__global__ void __launch_bounds__(AD_THREADS) k_force_allpairs_dotf(Params<float> p, State<float> s, AllPairsDotF a,
                                                                    Force<float> f, EnergyOut eo)
{
    __shared__ Vec4<float> sj[AD_THREADS];               // one tile, two barriers per tile: the fp64 kernel's register
    __shared__ int sid[AD_THREADS];                      // prefetch + second buffer measured 4-6 % slower here
    const int base = blockIdx.x * (AD_THREADS * IB) + threadIdx.x;
    float ax[IB], ay[IB], az[IB];                          // 2 x_i, 2 y_i, 2 z_i
    Vec4<float> ro[IB];                                    // original positions, for the exact path
    int idx[IB], thr[IB];                                  // thr: bits of |r_i|^2 - (r_c^2 + rounding bound) > 0
#pragma unroll
    for (int b = 0; b < IB; ++b) {
        idx[b] = base + b * AD_THREADS;
        Vec4<float> e = {1.0e9f, 1.0e9f, 1.0e9f, -3.0e18f};
        ro[b] = e;
        if (idx[b] < p.nv) { e = a.jv[idx[b]]; ro[b] = s.r[idx[b]]; }
        ax[b] = 2.f * e.x; ay[b] = 2.f * e.y; az[b] = 2.f * e.z;
        thr[b] = __float_as_int(-e.w - a.thr);
    }
    Acc<float, ENERGY> av[IB], aw[IB];
    bool any = false;
    const bool px = p.bc[0] == BC_PERIODIC, py = p.bc[1] == BC_PERIODIC, pz = p.bc[2] == BC_PERIODIC;
    const int nvj = p.nv + *a.ghost_count;
    const int tiles_v = (nvj + AD_THREADS - 1) / AD_THREADS, tiles_w = (a.nwg + AD_THREADS - 1) / AD_THREADS;
    for (int t = blockIdx.y; t < tiles_v + tiles_w; t += gridDim.y) {
        const bool wall = t >= tiles_v;
        const int j0 = (wall ? t - tiles_v : t) * AD_THREADS;
        const int nj = wall ? a.nwg : nvj;
        __syncthreads();
        {
            Vec4<float> e = {-1.0e9f, -1.0e9f, -1.0e9f, -3.0e18f};
            int id = -1;
            if (j0 + threadIdx.x < nj) { e = (wall ? a.jw : a.jv)[j0 + threadIdx.x]; id = (wall ? a.jw_id : a.jv_id)[j0 + threadIdx.x]; }
            sj[threadIdx.x] = e;
            sid[threadIdx.x] = id;
        }
        __syncthreads();
        for (int k0 = 0; k0 < AD_THREADS; k0 += AD_UNROLL) {
            // positive floats order like their bits, a negative t is a negative integer (see the fp64 kernel)
            int top[IB];
#pragma unroll
            for (int b = 0; b < IB; ++b) top[b] = (int)0x80000000;
#pragma unroll
            for (int u = 0; u < AD_UNROLL; ++u) {
                const Vec4<float> q = sj[k0 + u];
#pragma unroll
                for (int b = 0; b < IB; ++b)
                    top[b] = max(top[b], __float_as_int(fmaf(ax[b], q.x, fmaf(ay[b], q.y, fmaf(az[b], q.z, q.w)))));
            }
            bool cand = false;
#pragma unroll
            for (int b = 0; b < IB; ++b) cand |= top[b] >= thr[b];
            if (cand) {
                for (int u = 0; u < AD_UNROLL; ++u) {
                    const Vec4<float> q = sj[k0 + u];
                    const int jo = sid[k0 + u];
#pragma unroll
                    for (int b = 0; b < IB; ++b) {
                        if (__float_as_int(fmaf(ax[b], q.x, fmaf(ay[b], q.y, fmaf(az[b], q.z, q.w)))) < thr[b]) continue;
                        if (jo < 0 || idx[b] >= p.nv || (!wall && jo == idx[b])) continue;
                        const Vec4<float> rj = wall ? a.wr[jo] : s.r[jo];
                        float dx = ro[b].x - rj.x, dy = ro[b].y - rj.y, dz = ro[b].z - rj.z;
                        if (px) dx = min_image(ro[b].x, rj.x, dx, p.L[0], p.invL[0]);
                        if (py) dy = min_image(ro[b].y, rj.y, dy, p.L[1], p.invL[1]);
                        if (pz) dz = min_image(ro[b].z, rj.z, dz, p.L[2], p.invL[2]);
                        if (wall) pair_term<float, ENERGY>(dx, dy, dz, p.rc2, p.sig2_vw, p.e24_vw, p.e4_vw, p.uc_vw, aw[b]);
                        else pair_term<float, ENERGY>(dx, dy, dz, p.rc2, p.sig2_vv, p.e24_vv, p.e4_vv, p.uc_vv, av[b]);
                    }
                }
                any = true;
            }
        }
    }
    if (!any) return;
#pragma unroll
    for (int b = 0; b < IB; ++b) {
        const int i = idx[b];
        if (i >= p.nv) continue;
        const float fx = av[b].fx + aw[b].fx, fy = av[b].fy + aw[b].fy, fz = av[b].fz + aw[b].fz;
        if (!ENERGY) {
            if (fx != 0.f || fy != 0.f || fz != 0.f) { atomicAdd(&f.fx[i], fx); atomicAdd(&f.fy[i], fy); atomicAdd(&f.fz[i], fz); }
        } else if (av[b].c | aw[b].c) {
            atomicAdd(&eo.pe[i], 0.5 * av[b].u + aw[b].u);
            atomicAdd(&eo.pew[i], aw[b].u);
            atomicAdd(&eo.vir[i], 0.5 * av[b].w + aw[b].w);
            atomicAdd(&eo.cvv[i], av[b].c);
            atomicAdd(&eo.cvw[i], aw[b].c);
        }
    }
}

} // namespace md
