// md_api.cu -- C ABI (include/md.h) over the kernels in md_kernels.cuh.
// Host logic only: validation, workspace carving, launch order, CUDA graphs.
#include "../../include/md.h"
#include "md_kernels.cuh"
#include "md_verlet.cuh"
#include "md_allpairs.cuh"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <type_traits>
#include <algorithm>
#include <vector>

namespace {

thread_local std::string g_create_error;

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
inline int cdiv(long long a, long long b) { return (int)((a + b - 1) / b); }

// Bump allocator over the caller's workspace; base == nullptr only measures.
struct Carver {
    char* base;
    size_t off = 0;
    explicit Carver(void* b) : base((char*)b) {}
    template <typename U>
    U* take(size_t n)
    {
        off = align_up(off, 256);
        U* p = base ? (U*)(base + off) : nullptr;
        off += n * sizeof(U);
        return p;
    }
};

struct GridSpec {
    int nc[3];
    long long ncell;
    bool cells_ok;
};

GridSpec make_grid(const md_box& box, double rc)
{
    GridSpec g;
    g.cells_ok = true;
    g.ncell = 1;
    for (int a = 0; a < 3; ++a) {
        g.nc[a] = 1;
        if (a < box.dim) {
            int k = (int)std::floor(box.len[a] / rc);
            if (k < 1) k = 1;
            if (box.bc[a] == MD_BC_PERIODIC && k < 3) g.cells_ok = false;
            g.nc[a] = k;
        }
        g.ncell *= g.nc[a];
    }
    if (g.ncell > (1ll << 30)) g.cells_ok = false;
    return g;
}

const char* validate(const md_box* box, const md_lj* lj, const md_opts* o, long long nv, long long nw)
{
    if (!box || !lj || !o) return "null parameter struct";
    if (box->dim != 2 && box->dim != 3) return "dim must be 2 or 3";
    if (nv < 1 || nv > (1ll << 30)) return "n_vapor must be in [1, 2^30]";
    if (nw < 0 || nw > (1ll << 30)) return "n_wall must be in [0, 2^30]";
    if (!(o->dt > 0) || !std::isfinite(o->dt)) return "dt must be > 0";
    if (!(o->mass > 0) || !std::isfinite(o->mass)) return "mass must be > 0";
    if (o->precision != 64 && o->precision != 32) return "precision must be 64 or 32";
    if (o->force_algo < MD_FORCE_AUTO || o->force_algo > MD_FORCE_VERLET) return "unknown force_algo";
    if (!(o->skin >= 0) || !std::isfinite(o->skin)) return "skin must be >= 0";
    if (o->skin >= lj->r_cut) return "skin must be < r_cut";
    if (o->heavy_list < 0) return "heavy_list must be >= 0";
    if (o->list_prunes > 8) return "list_prunes must be <= 8";
    if (!std::isfinite(o->tau_b) || !std::isfinite(o->t_target)) return "tau_b, t_target must be finite";
    if (o->tau_b > 0 && (o->tau_b < o->dt || !(o->t_target > 0))) return "thermostat needs tau_b >= dt and t_target > 0";
    if (!(lj->r_cut > 0) || !std::isfinite(lj->r_cut)) return "r_cut must be > 0";
    if (!(lj->sigma > 0) || !(lj->sigma_w > 0)) return "sigma, sigma_w must be > 0";
    if (!std::isfinite(lj->eps) || !std::isfinite(lj->eps_w)) return "eps, eps_w must be finite";
    for (int a = 0; a < box->dim; ++a) {
        if (!(box->len[a] > 0) || !std::isfinite(box->len[a])) return "box length must be > 0";
        if (box->bc[a] != MD_BC_PERIODIC && box->bc[a] != MD_BC_REFLECT) return "unknown boundary condition";
        if (box->bc[a] == MD_BC_PERIODIC && box->len[a] < 2.0 * lj->r_cut)
            return "periodic box length < 2 r_cut (minimum image undefined)";
    }
    return nullptr;
}

double list_skin(const md_lj& lj, const md_opts& o) { return o.skin > 0 ? o.skin : 0.24 * lj.r_cut; }

// Two-level list: k prunes between two full rebuilds need an outer skin of (k + 1) skins -- each list event is raised when
// a path exceeds skin / 2 -- plus a margin for the step that crosses the threshold (a prune that finds a longer path is
// discarded, so the margin is a matter of speed, not of correctness).
double outer_skin(double skin, int k) { return k > 0 ? (k + 1) * skin * 1.07 : skin; }

// Prunes per full rebuild: md_opts.list_prunes (0: two; < 0: none), reduced until the box holds >= 3 cells of side
// r_cut + outer skin in every periodic dimension.
int resolve_prunes(const md_box& box, const md_lj& lj, const md_opts& o)
{
    int k = o.list_prunes > 0 ? std::min(o.list_prunes, 8) : (o.list_prunes == 0 ? 2 : 0);
    const double skin = list_skin(lj, o);
    for (; k > 0; --k) {
        bool ok = make_grid(box, lj.r_cut + outer_skin(skin, k)).cells_ok;
        for (int a = 0; a < box.dim; ++a)
            if (box.bc[a] == MD_BC_PERIODIC && box.len[a] <= 2.0 * (lj.r_cut + outer_skin(skin, k))) ok = false;
        if (ok) break;
    }
    return k;
}

// Grid the handle uses: cells of side >= r_cut (CELLS) or >= r_cut + (outer) skin (VERLET).
GridSpec grid_for(const md_box& box, const md_lj& lj, const md_opts& o, int algo)
{
    return make_grid(box, algo == MD_FORCE_VERLET ? lj.r_cut + outer_skin(list_skin(lj, o), resolve_prunes(box, lj, o)) : lj.r_cut);
}

bool verlet_ok(const md_box& box, const md_lj& lj, const md_opts& o, long long nv, long long nw)
{
    const double rl = lj.r_cut + list_skin(lj, o);
    for (int a = 0; a < box.dim; ++a)
        if (box.bc[a] == MD_BC_PERIODIC && box.len[a] <= 2.0 * rl) return false;
    return make_grid(box, rl).cells_ok && nv + nw < (1ll << 30);
}

int pick_algo(const md_box& box, const md_lj& lj, const md_opts& o, long long nv, long long nw)
{
    const bool cells_ok = make_grid(box, lj.r_cut).cells_ok;
    if (o.force_algo == MD_FORCE_ALLPAIRS) return MD_FORCE_ALLPAIRS;
    if (o.force_algo == MD_FORCE_CELLS) return cells_ok ? MD_FORCE_CELLS : -1;
    if (o.force_algo == MD_FORCE_VERLET) return verlet_ok(box, lj, o, nv, nw) ? MD_FORCE_VERLET : -1;
    // AUTO: the fastest valid path (measured on every configuration, profiles/r01_report_all_configs.md)
    if (verlet_ok(box, lj, o, nv, nw)) return MD_FORCE_VERLET;
    return cells_ok ? MD_FORCE_CELLS : MD_FORCE_ALLPAIRS;
}

template <typename T>
struct Layout {
    md::State<T> st[2];
    md::Force<T> f;
    int *cell, *slot, *count, *start, *tile_sum;
    unsigned long long* tile_agg;   // VERLET: in-kernel scan's published tile sums
    md::Vec4<T> *wr, *wtr;      // wall positions: cell order / caller's order
    int *wcell, *wslot, *wstart;
    uint8_t* wnear;
    md::EnergyOut eo;
    double *part, *eout;
    int* err;
    unsigned long long* tests;
    double *stage0, *stage1, *wstage;
    int *nbr, *ncnt, *vflags;   // VERLET: neighbour list, counts, flags
    int *onbr, *ocnt, *oheavy;  // VERLET, two-level list: outer list, its counts, particles pruned by a warp
    T* wo;                      // path between the last full rebuild and the last list event
    unsigned long long* vtimes;
    unsigned long long* vbar;   // VERLET: grid-barrier arrival counter
    md::F4* r32;                // VERLET fp64: fp32 shadow of the positions for the list build
    unsigned long long* hist;   // density-profile bins
    double* vksum;              // VERLET thermostat: rotating kinetic-energy accumulators
    md::Vec4<T> *jv, *jw;       // ALLPAIRS: j lists (entries + ghosts) of the dot-product kernels
    int *jv_id, *jw_id;         // fp32: original index of every entry
    int* ghost_count;
    int red_blocks;
    size_t bytes;
};

// Image blocks of a VERLET position buffer (md_verlet.cuh): bit a of the block number = shifted in dimension a, so
// the count is 1 + the sum of the periodic dimensions' bits; fp32 mode keeps block 0 only (it folds differences).
int image_blocks(const md_box& box, int precision)
{
    int top = 0;
    if (precision == 64)
        for (int a = 0; a < box.dim; ++a)
            if (box.bc[a] == MD_BC_PERIODIC) top |= 1 << a;
    return top + 1;
}

template <typename T>
Layout<T> carve(void* base, int dim, long long nv, long long nw, long long ncell, int algo, int nimg, int nprune)
{
    Layout<T> l;
    Carver c(base);
    const bool cells = algo != MD_FORCE_ALLPAIRS, verlet = algo == MD_FORCE_VERLET;
    size_t n = (size_t)align_up((size_t)nv, 64);
    size_t m = (size_t)align_up((size_t)(nw > 0 ? nw : 1), 64);
    for (int b = 0; b < (cells ? 2 : 1); ++b) {
        // VERLET: nimg image blocks of nv + nw entries each (walls appended at [nv, nv + nw) of every block)
        l.st[b].r = c.take<md::Vec4<T>>(verlet ? (size_t)nimg * (size_t)(nv + nw) + 64 : n);
        l.st[b].vx = c.take<T>(n); l.st[b].vy = c.take<T>(n); l.st[b].vz = c.take<T>(n);
        l.st[b].id = c.take<int>(n);
    }
    if (!cells) l.st[1] = l.st[0];
    l.f.fx = c.take<T>(n); l.f.fy = c.take<T>(n); l.f.fz = c.take<T>(n);
    l.cell = c.take<int>(n > m ? n : m);
    l.slot = c.take<int>(n > m ? n : m);
    size_t nc = cells ? (size_t)ncell : 1;
    l.count = c.take<int>(nc);
    l.start = c.take<int>(nc + 1);
    l.tile_sum = c.take<int>((size_t)cdiv((long long)nc, md::SCAN_TILE) + 1);
    l.wr = c.take<md::Vec4<T>>(m);
    l.wtr = c.take<md::Vec4<T>>(m);
    l.wcell = l.cell; l.wslot = l.slot;   // wall binning runs once, before the vapor's
    l.wstart = c.take<int>(nc + 1);
    l.wnear = c.take<uint8_t>(nc);
    l.eo.pe = c.take<double>(n); l.eo.pew = c.take<double>(n); l.eo.vir = c.take<double>(n);
    l.eo.cvv = c.take<int>(n); l.eo.cvw = c.take<int>(n);
    l.red_blocks = (int)std::min<long long>(cdiv(nv, md::RED_THREADS), 1024);
    l.part = c.take<double>(6 * (size_t)l.red_blocks);
    l.eout = c.take<double>(8);
    l.err = c.take<int>(4);
    l.tests = c.take<unsigned long long>(2);
    l.nbr = c.take<int>(verlet ? n * md::VL_MAXN : 1);
    l.ncnt = c.take<int>(verlet ? n : 1);
    const bool two = verlet && nprune > 0;
    l.onbr = c.take<int>(two ? n * md::VL_MAXO : 1);
    l.ocnt = c.take<int>(two ? n : 1);
    l.oheavy = c.take<int>(two ? n : 1);
    l.wo = c.take<T>(two ? n : 1);
    l.vflags = c.take<int>(md::VF_COUNT);
    l.r32 = c.take<md::F4>(verlet && sizeof(T) == 8 ? n + m : 1);
    l.tile_agg = c.take<unsigned long long>(verlet ? (size_t)cdiv((long long)nc, md::SCAN_TILE) + 1 : 1);
    const bool dot = algo == MD_FORCE_ALLPAIRS;
    l.jv = c.take<md::Vec4<T>>(dot ? 8 * n : 1);          // <= 7 periodic images per particle
    l.jw = c.take<md::Vec4<T>>(dot ? 8 * m : 1);
    l.jv_id = c.take<int>(dot && sizeof(T) == 4 ? 8 * n : 1);
    l.jw_id = c.take<int>(dot && sizeof(T) == 4 ? 8 * m : 1);
    l.ghost_count = c.take<int>(4);
    l.vtimes = c.take<unsigned long long>(16 + 8192);
    l.vbar = c.take<unsigned long long>(2);
    l.vksum = c.take<double>(4);
    l.hist = c.take<unsigned long long>(md::HIST_MAX_BINS);
    l.stage0 = c.take<double>(n * dim);
    l.stage1 = c.take<double>(n * dim);
    l.wstage = c.take<double>(m * dim);
    l.bytes = align_up(c.off, 256);
    return l;
}

} // namespace

struct md_sim {
    std::string err;
    virtual ~md_sim() {}
    virtual int step(long long n) = 0;
    virtual int get_state(double* pos, double* vel, double* force, double* pe, long long* step) = 0;
    virtual int energy(md_energy_out* out) = 0;
    virtual int profile(long long n, md_kernel_times* out) = 0;
    virtual int pair_tests(long long* tests) = 0;
    virtual void info(int* algo, int nc[3], int* kps) const = 0;
    virtual int pressure(md_pressure_out* out) = 0;
    virtual int density(int n_axial, long long* axial, int n_radial, double r_max, long long* radial) = 0;
    virtual void drain() = 0;
    md_pore pore = {};
    md_box box = {};
};

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) {                                                                   \
            err = std::string(#call) + ": " + cudaGetErrorString(e_);                              \
            return MD_ERR_CUDA;                                                                    \
        }                                                                                          \
    } while (0)

namespace {

template <typename T>
struct Sim : md_sim {
    md::Params<T> p;
    Layout<T> l;
    md::Walls<T> walls;
    int dim = 3, algo = MD_FORCE_CELLS, cur = 0;
    long long step_no = 0, energy_step = -1;
    cudaStream_t stream = nullptr;
    cudaGraphExec_t g1[2] = {nullptr, nullptr}, gN[2] = {nullptr, nullptr};
    static constexpr int CHUNK = 16;
    cudaEvent_t ev[5] = {};
    double e_host[6];
    // VERLET (persistent kernel): device-side buffer parities are mirrored here by refresh()
    md::Verlet<T> vl;
    int curv = 0, coop_grid = 0, coop_base = 0, coop_max = 0, heavy_seen = 0, heavy32_seen = 0;
    int minb3_threshold = -1;   // particles beyond which the 3-blocks-per-SM build runs; set at the first launch
    long long rebuilds_seen = 0, prunes_seen = 0;
    unsigned long long phase_ns[10] = {};

    md::AllPairsDot ad;
    md::AllPairsDotF adf;
    bool dot = false;           // all-pairs through the dot-product kernels (md_allpairs.cuh)
    int ad_slices = 1, ad_ib = md::AD_IB;
    int gpar = 0;               // which of the two ghost counters describes the current j list

    bool verlet() const { return algo == MD_FORCE_VERLET; }
    void drain() override { cudaStreamSynchronize(stream); }

    // Particle state as the post-processing kernels see it (positions from `cur`, the rest from `curv`).
    md::State<T> view() const
    {
        md::State<T> s = l.st[verlet() ? curv : cur];
        s.r = l.st[cur].r;
        return s;
    }

    int launch_run(long long n, int force_rebuild)
    {
#ifdef MD_DIAGNOSTICS
        if (minb3_threshold < 0 && getenv("MD_MINB3_THRESHOLD")) minb3_threshold = atoi(getenv("MD_MINB3_THRESHOLD"));
#endif
        if (minb3_threshold < 0) {
            // Two resident blocks per SM (128 registers, state carried in registers across the barrier) while the
            // particles fit that grid with one thread each; beyond it three blocks of the 80-register variant:
            // measured 13.4 vs 18.0 us per step at N = 80,000, 21.0 vs 23.9 at 2^17, 31.6 vs 34.4 at 2^18, 104 vs
            // 127 at 2^20, and 12.1 vs 11.9 at 2^16 (profiles/r01_heavy_groups.md)
            int dev = 0, sms = 0;
            CK(cudaGetDevice(&dev));
            CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
            minb3_threshold = 2 * sms * md::VL_THREADS;
        }
        const bool big = p.nv > minb3_threshold;
        void* kernel = dim == 3 ? (big ? (void*)md::k_md_run<T, 9, 3> : (void*)md::k_md_run<T, 9, 2>)
                                : (big ? (void*)md::k_md_run<T, 3, 3> : (void*)md::k_md_run<T, 3, 2>);
        if (!coop_max) {
            int dev = 0, sms = 0, coop = 0, nb = 0;
            CK(cudaGetDevice(&dev));
            CK(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
            if (!coop) { err = "device does not support cooperative launches"; return MD_ERR_UNSUPPORTED; }
            CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
            CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kernel, md::VL_THREADS, 0));
            if (nb < 1) { err = "persistent kernel does not fit on an SM"; return MD_ERR_CUDA; }
            coop_max = nb * sms;
            // one thread per particle; whole multiples of the SM count keep the SMs evenly loaded
            const int want = cdiv(cdiv(p.nv, md::VL_THREADS), sms) * sms;
            coop_base = std::max(1, std::min(coop_max, p.nv <= md::VL_THREADS * sms ? cdiv(p.nv, md::VL_THREADS) : want));
        }
        // Blocks past the last particle serve the lane groups of the particles with long lists (the kernel hands
        // out only as many as those blocks hold: measured -13 % per step at 2^16 with them, +1..2 % at 2^18 and
        // 2^20 where the work would land on busy blocks, profiles/r01_heavy_groups.md): an eighth of the particle
        // blocks, or what the last list this handle has seen asked for (refresh() mirrors the counts) plus a quarter:
        // four lanes per long list, a warp per VL_WARP_ROUNDS very long ones.
        const int light = cdiv(p.nv, md::VL_THREADS);
        coop_grid = coop_base;
        if (light < coop_max) {
            const int idle4 = cdiv(heavy_seen * md::VL_GROUP * 5 / 4, md::VL_THREADS);
            const int idle32 = cdiv(heavy32_seen * 5 / 4, md::VL_WARP_ROUNDS * (md::VL_THREADS / 32));
            coop_grid = std::min(coop_max, std::max(coop_base, light + std::max(light / 8, std::max(idle4, idle32)) + 1));
        }
        CK(cudaMemsetAsync(l.vbar, 0, 2 * sizeof(unsigned long long), stream));        // grid barrier counter
        CK(cudaMemsetAsync(l.vksum, 0, 4 * sizeof(double), stream));
        void* args[] = {(void*)&p, (void*)&vl, (void*)&n, (void*)&force_rebuild};
        CK(cudaLaunchCooperativeKernel(kernel, dim3(coop_grid), dim3(md::VL_THREADS), args, 0, stream));
        return MD_OK;
    }

    // Synchronises and mirrors the persistent kernel's flags; reports its error flags.
    int refresh()
    {
        if (!verlet()) return MD_OK;
        int h[md::VF_COUNT];
        CK(cudaMemcpyAsync(h, l.vflags, sizeof(h), cudaMemcpyDeviceToHost, stream));
        CK(cudaStreamSynchronize(stream));
        CK(cudaGetLastError());
        cur = h[md::VF_CUR]; curv = h[md::VF_CURV]; rebuilds_seen = h[md::VF_NREBUILD]; prunes_seen = h[md::VF_NPRUNE];
        heavy_seen = h[md::VF_NHEAVY + h[md::VF_HPAR]]; heavy32_seen = h[md::VF_NHEAVY32 + h[md::VF_HPAR]];
        if (h[md::VF_ESCAPE]) { err = "a particle left a reflecting box (more than one bounce in a step)"; return MD_ERR_STATE; }
        if (h[md::VF_OVERFLOW]) { err = "neighbour list overflow (> 128 neighbours within r_cut + skin)"; return MD_ERR_WORKSPACE; }
        return MD_OK;
    }

    ~Sim() override
    {
        for (int k = 0; k < 2; ++k) {
            if (g1[k]) cudaGraphExecDestroy(g1[k]);
            if (gN[k]) cudaGraphExecDestroy(gN[k]);
        }
        for (auto& e : ev) if (e) cudaEventDestroy(e);
    }

    int blocks(int threads) const { return cdiv(p.nv, threads); }

    // ---- a2: bin `n` particles of state s into cell order (count -> scan -> caller scatters)
    void launch_scan(int* count, int* start)
    {
        int tiles = cdiv(p.ncell, md::SCAN_TILE);
        md::k_scan_reduce<<<tiles, md::SCAN_THREADS, 0, stream>>>(count, p.ncell, l.tile_sum);
        md::k_scan_apply<<<tiles, md::SCAN_THREADS, 0, stream>>>(count, p.ncell, l.tile_sum, start);
    }

    template <bool ENERGY, bool KICK, bool COUNT>
    void launch_force()
    {
        if (verlet()) {
            if (ENERGY)
                md::k_verlet_energy<T><<<cdiv(p.nv, md::VL_THREADS), md::VL_THREADS, 0, stream>>>(
                    p, vl, cur, l.eo);
        } else if (algo == MD_FORCE_CELLS) {
            // ROWS lanes per particle: 9 in 3D (3 particles per warp), 3 in 2D (10 per warp)
            if (dim == 3)
                md::k_force_cells<T, 9, ENERGY, KICK, COUNT><<<cdiv(cdiv(p.nv, 3), 4), 128, 0, stream>>>(
                    p, l.st[cur], l.start, walls, l.f, l.eo, l.tests);
            else
                md::k_force_cells<T, 3, ENERGY, KICK, COUNT><<<cdiv(cdiv(p.nv, 10), 4), 128, 0, stream>>>(
                    p, l.st[cur], l.start, walls, l.f, l.eo, l.tests);
        } else if (dot) {
            {
                ad.ghost_count = adf.ghost_count = l.ghost_count + gpar;
                if (ENERGY) {
                    const size_t n = (size_t)p.nv;
                    cudaMemsetAsync(l.eo.pe, 0, n * sizeof(double), stream);
                    cudaMemsetAsync(l.eo.pew, 0, n * sizeof(double), stream);
                    cudaMemsetAsync(l.eo.vir, 0, n * sizeof(double), stream);
                    cudaMemsetAsync(l.eo.cvv, 0, n * sizeof(int), stream);
                    cudaMemsetAsync(l.eo.cvw, 0, n * sizeof(int), stream);
                }
                const dim3 grid(cdiv(p.nv, md::AD_THREADS * ad_ib), ad_slices);
                if constexpr (std::is_same<T, double>::value) {
                    if (ad_ib == 1) md::k_force_allpairs_dot<ENERGY, 1><<<grid, md::AD_THREADS, 0, stream>>>(p, ad, l.f, l.eo);
                    else md::k_force_allpairs_dot<ENERGY, md::AD_IB><<<grid, md::AD_THREADS, 0, stream>>>(p, ad, l.f, l.eo);
                } else {
                    if (ad_ib == 1) md::k_force_allpairs_dotf<ENERGY, 1><<<grid, md::AD_THREADS, 0, stream>>>(p, l.st[cur], adf, l.f, l.eo);
                    else md::k_force_allpairs_dotf<ENERGY, md::AD_IB><<<grid, md::AD_THREADS, 0, stream>>>(p, l.st[cur], adf, l.f, l.eo);
                }
                // the second half-kick also clears the OTHER ghost counter, which the next step's list will fill
                if (KICK) md::k_ap_kick<T><<<blocks(256), 256, 0, stream>>>(p, l.st[cur], l.f, l.ghost_count + (gpar ^ 1));
            }
        } else
            md::k_force_allpairs<T, ENERGY, KICK><<<blocks(md::AP_THREADS), md::AP_THREADS, 0, stream>>>(
                p, l.st[cur], l.wtr, l.f, l.eo);
    }

    // One velocity-Verlet step: a1 -> a2 -> a3 + a4. `t` (optional) = events around each kernel.
    void enqueue_step(cudaEvent_t* t)
    {
        if (t) cudaEventRecord(t[0], stream);
        if (algo == MD_FORCE_CELLS) {
            md::k_kick_drift_bin<T, true, true><<<blocks(256), 256, 0, stream>>>(p, l.st[cur], l.f, l.count, l.cell,
                                                                                l.slot, l.err);
            if (t) cudaEventRecord(t[1], stream);
            launch_scan(l.count, l.start);
            if (t) cudaEventRecord(t[2], stream);
            md::k_scatter<T><<<blocks(256), 256, 0, stream>>>(p.nv, l.st[cur], l.st[cur ^ 1], l.f, l.f, l.cell, l.slot,
                                                              l.start, 0);
            cur ^= 1;
            if (t) cudaEventRecord(t[3], stream);
        } else {
            if (dot) {
                gpar ^= 1;
                ad.ghost_count = adf.ghost_count = l.ghost_count + gpar;
                if constexpr (std::is_same<T, double>::value)
                    md::k_ap_kick_drift_list<true><<<blocks(256), 256, 0, stream>>>(p, l.st[cur], l.f, ad, l.err);
                else
                    md::k_apf_kick_drift_list<true><<<blocks(256), 256, 0, stream>>>(p, l.st[cur], l.f, adf, l.err);
            } else
                md::k_kick_drift_bin<T, true, false><<<blocks(256), 256, 0, stream>>>(p, l.st[cur], l.f, nullptr, nullptr,
                                                                                     nullptr, l.err);
            if (t) { cudaEventRecord(t[1], stream); cudaEventRecord(t[2], stream); cudaEventRecord(t[3], stream); }
        }
        launch_force<false, true, false>();
        if (p.thermo_rate > 0.0) {   // F4: K partial sums, then lambda + rescale
            md::k_kinetic_partial<T><<<l.red_blocks, md::RED_THREADS, 0, stream>>>(p.nv, p.mass, l.st[cur], l.part);
            md::k_thermo_scale<T><<<blocks(256), 256, 0, stream>>>(p, l.st[cur], l.red_blocks, l.part);
        }
        if (t) cudaEventRecord(t[4], stream);
    }

    int capture(int nsteps, cudaGraphExec_t* out)
    {
        cudaGraph_t g = nullptr;
        CK(cudaStreamBeginCapture(stream, cudaStreamCaptureModeThreadLocal));
        for (int k = 0; k < nsteps; ++k) enqueue_step(nullptr);
        CK(cudaStreamEndCapture(stream, &g));
        cudaError_t e = cudaGraphInstantiate(out, g, 0);
        cudaGraphDestroy(g);
        if (e != cudaSuccess) { err = std::string("cudaGraphInstantiate: ") + cudaGetErrorString(e); return MD_ERR_CUDA; }
        return MD_OK;
    }

    int step(long long n) override
    {
        if (n < 0) { err = "n_steps < 0"; return MD_ERR_INVALID_ARG; }
        if (verlet()) {
            if (n == 0) return MD_OK;
            int rc = launch_run(n, 0);
            if (rc == MD_OK) step_no += n;
            return rc;
        }
        if (stream == nullptr || stream == cudaStreamLegacy || stream == cudaStreamPerThread) {
            // the default streams cannot be captured: plain launches
            for (long long k = 0; k < n; ++k) enqueue_step(nullptr);
            step_no += n;
            CK(cudaGetLastError());
            return MD_OK;
        }
        while (n > 0) {
            const int par = algo == MD_FORCE_CELLS ? cur : (dot ? gpar : 0);
            if (n >= CHUNK) {
                if (!gN[par]) { int c0 = cur, g0 = gpar; int rc = capture(CHUNK, &gN[par]); cur = c0; gpar = g0; if (rc) return rc; }
                CK(cudaGraphLaunch(gN[par], stream));
                n -= CHUNK; step_no += CHUNK;       // CHUNK is even: buffer parity unchanged
            } else {
                if (!g1[par]) { int c0 = cur, g0 = gpar; int rc = capture(1, &g1[par]); cur = c0; gpar = g0; if (rc) return rc; }
                CK(cudaGraphLaunch(g1[par], stream));
                if (algo == MD_FORCE_CELLS) cur ^= 1;
                if (dot) { gpar ^= 1; ad.ghost_count = adf.ghost_count = l.ghost_count + gpar; }
                n -= 1; step_no += 1;
            }
        }
        return MD_OK;
    }

    int profile(long long n, md_kernel_times* out) override
    {
        if (!out || n < 0) { err = "bad arguments"; return MD_ERR_INVALID_ARG; }
        memset(out, 0, sizeof(*out));
        for (auto& e : ev) if (!e) CK(cudaEventCreate(&e));
        if (verlet()) {
            int rc = refresh();
            if (rc) return rc;
            const long long r0 = rebuilds_seen, p0 = prunes_seen;
            unsigned long long t[10], tb[10];                 // the kernel's own timers are cumulative: take the difference
            CK(cudaMemcpy(tb, l.vtimes, sizeof(tb), cudaMemcpyDeviceToHost));
            CK(cudaEventRecord(ev[0], stream));
            if (n > 0 && (rc = launch_run(n, 0))) return rc;
            CK(cudaEventRecord(ev[1], stream));
            if ((rc = refresh())) return rc;
            float ms = 0.f;
            CK(cudaEventElapsedTime(&ms, ev[0], ev[1]));
            CK(cudaMemcpy(t, l.vtimes, sizeof(t), cudaMemcpyDeviceToHost));
#ifdef MD_DIAGNOSTICS
            if (getenv("MD_DEBUG_TIMES")) {
                std::vector<unsigned long long> w(8192);
                CK(cudaMemcpy(w.data(), l.vtimes + 16, 8192 * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
                const int nwarp = coop_grid * md::VL_THREADS / 32;
                const int nbl = std::min(coop_grid, cdiv(p.nv, md::VL_THREADS)), wpb = md::VL_THREADS / 32;
                double mx[2] = {0, 0}, sm[2] = {0, 0};
                int cnt[2] = {0, 0};
                for (int k = 0; k < nwarp && k < 8192; ++k) {
                    const int g = k / wpb >= nbl;
                    mx[g] = std::max(mx[g], (double)w[k]); sm[g] += (double)w[k]; ++cnt[g];
                }
                const double per = 1e-3 / std::max<long long>(step_no + n, 1);
                fprintf(stderr, "[md] step-phase us per step and warp (cumulative / steps): particle blocks (%d) max %.2f mean %.2f | idle blocks (%d) max %.2f mean %.2f\n",
                        nbl, mx[0] * per, sm[0] * per / std::max(cnt[0], 1), coop_grid - nbl, mx[1] * per, sm[1] * per / std::max(cnt[1], 1));
                {
                    double l = 0, h = 0, ml = 0, mh = 0;
                    for (int k = 0; k < 1024; ++k) {
                        l += (double)w[4096 + 2 * k]; h += (double)w[4097 + 2 * k];
                        ml = std::max(ml, (double)w[4096 + 2 * k]); mh = std::max(mh, (double)w[4097 + 2 * k]);
                    }
                    const double np = std::max<double>((double)prunes_seen, 1.0);
                    fprintf(stderr, "[md] prune, us per prune and warp (first 1024 warps): thread-per-particle part mean %.2f max %.2f, "
                            "warp-per-particle part mean %.2f max %.2f; particles pruned by warps: %.0f per prune; histogram of step-phase times (1.024 us bins):",
                            l / 1024 / np * 1e-3, ml / np * 1e-3, h / 1024 / np * 1e-3, mh / np * 1e-3, (double)w[7000] / np);
                    for (int k = 0; k < 16; ++k) fprintf(stderr, " %llu", w[8000 + k]);
                    fprintf(stderr, "\n");
                }
                int hh[md::VF_COUNT];
                CK(cudaMemcpy(hh, l.vflags, sizeof(hh), cudaMemcpyDeviceToHost));
                fprintf(stderr, "[md] after the last rebuild: lists > %d entries %d (lane groups hold %d), lists > %d entries %d (warps hold %d)\n",
                        vl.heavy_t, hh[md::VF_NHEAVY + hh[md::VF_HPAR]], hh[md::VF_HCAP], md::VL_WARP_T, hh[md::VF_NHEAVY32 + hh[md::VF_HPAR]], hh[md::VF_HCAP32]);
            }
#endif
            for (int q = 0; q < 10; ++q) phase_ns[q] = t[q] - tb[q];
            out->prunes = prunes_seen - p0; out->prune_ms = phase_ns[8] * 1e-6;
            for (int q = 0; q < 4; ++q) out->rebuild_ms[q] = phase_ns[4 + q] * 1e-6;   // bin, scan, scatter, list build
            // VERLET: ms[0] step phases, ms[1] grid barriers, ms[2] rebuilds (as seen by thread 0), ms[3] whole launch
            out->ms[0] = phase_ns[0] * 1e-6; out->ms[1] = phase_ns[1] * 1e-6; out->ms[2] = phase_ns[2] * 1e-6;
            out->ms[3] = out->total_ms = ms;
            out->launches[3] = n > 0 ? 1 : 0;
            out->steps = n; out->rebuilds = rebuilds_seen - r0;
            step_no += n;
#ifdef MD_DIAGNOSTICS
            if (getenv("MD_DEBUG_BUILD")) {      // the build and force phases as kernels of their own, for ncu
                for (int k = 0; k < 3; ++k) {
                    if (dim == 3) md::k_dbg_build<T, 9><<<coop_grid, md::VL_THREADS, 0, stream>>>(p, vl, cur);
                    else md::k_dbg_build<T, 3><<<coop_grid, md::VL_THREADS, 0, stream>>>(p, vl, cur);
                }
                for (int k = 0; k < 3; ++k) md::k_dbg_force<T><<<coop_grid, md::VL_THREADS, 0, stream>>>(p, vl, cur, curv);
                if (vl.nprune > 0)      // leaves the handle unusable for further steps (heavy registries not refilled): last call only
                    for (int k = 0; k < 3; ++k) md::k_dbg_prune<T><<<coop_grid, md::VL_THREADS, 0, stream>>>(p, vl, cur);
                CK(cudaStreamSynchronize(stream));
            }
#endif
            return MD_OK;
        }
        for (long long k = 0; k < n; ++k) {
            enqueue_step(ev);
            CK(cudaStreamSynchronize(stream));
            for (int q = 0; q < 4; ++q) {
                float ms = 0.f;
                CK(cudaEventElapsedTime(&ms, ev[q], ev[q + 1]));
                out->ms[q] += ms;
            }
            float tot = 0.f;
            CK(cudaEventElapsedTime(&tot, ev[0], ev[4]));
            out->total_ms += tot;
            ++step_no;
        }
        const bool cells = algo == MD_FORCE_CELLS;
        out->launches[0] = n; out->launches[1] = cells ? 2 * n : 0; out->launches[2] = cells ? n : 0;
        out->launches[3] = n; out->steps = n;
        return MD_OK;
    }

    int check_err_flag()
    {
        if (verlet()) return refresh();
        int h = 0;
        CK(cudaMemcpyAsync(&h, l.err, sizeof(int), cudaMemcpyDeviceToHost, stream));
        CK(cudaStreamSynchronize(stream));
        if (h) { err = "a particle left a reflecting box (more than one bounce in a step)"; return MD_ERR_STATE; }
        return MD_OK;
    }

    int energy_pass()
    {
        if (energy_step == step_no) return MD_OK;
        launch_force<true, false, false>();
        md::k_energy_partial<T><<<l.red_blocks, md::RED_THREADS, 0, stream>>>(p.nv, p.mass, view(), l.eo, l.part);
        md::k_energy_final<<<1, md::RED_THREADS, 0, stream>>>(l.red_blocks, l.part, l.eout);
        CK(cudaMemcpyAsync(e_host, l.eout, 6 * sizeof(double), cudaMemcpyDeviceToHost, stream));
        CK(cudaStreamSynchronize(stream));
        CK(cudaGetLastError());
        energy_step = step_no;
        return MD_OK;
    }

    int energy(md_energy_out* out) override
    {
        if (!out) { err = "out is NULL"; return MD_ERR_INVALID_ARG; }
        int rc = check_err_flag();
        if (rc) return rc;
        rc = energy_pass();
        if (rc) return rc;
        out->kinetic = e_host[0];
        out->potential = e_host[1];
        out->potential_vw = e_host[2];
        out->potential_vv = e_host[1] - e_host[2];
        out->virial = e_host[3];
        out->pairs_vv = (long long)llround(e_host[4]) / 2;
        out->pairs_vw = (long long)llround(e_host[5]);
        out->step = step_no;
        if (!std::isfinite(out->kinetic) || !std::isfinite(out->potential)) {
            err = "non-finite energy";
            return MD_ERR_NONFINITE;
        }
        return MD_OK;
    }

    int export3(const T* a, const T* b, const T* c, double* host)
    {
        md::k_export3<T><<<blocks(256), 256, 0, stream>>>(p.nv, dim, view().id, a, b, c, l.stage0);
        CK(cudaMemcpyAsync(host, l.stage0, sizeof(double) * (size_t)p.nv * dim, cudaMemcpyDeviceToHost, stream));
        CK(cudaStreamSynchronize(stream));
        return MD_OK;
    }

    int get_state(double* pos, double* vel, double* force, double* pe, long long* step) override
    {
        int rc = check_err_flag();
        if (rc) return rc;
        const md::State<T> s = view();
        if (pos) {
            if (verlet()) md::k_export_pos_wrapped<T><<<blocks(256), 256, 0, stream>>>(p, dim, s.id, s.r, l.stage0);
            else md::k_export_pos<T><<<blocks(256), 256, 0, stream>>>(p.nv, dim, s.id, s.r, l.stage0);
            CK(cudaMemcpyAsync(pos, l.stage0, sizeof(double) * (size_t)p.nv * dim, cudaMemcpyDeviceToHost, stream));
            CK(cudaStreamSynchronize(stream));
        }
        if (vel && (rc = export3(s.vx, s.vy, s.vz, vel))) return rc;
        if (force && (rc = export3(l.f.fx, l.f.fy, l.f.fz, force))) return rc;
        if (pe) {
            if ((rc = energy_pass())) return rc;
            md::k_export1<<<blocks(256), 256, 0, stream>>>(p.nv, s.id, l.eo.pe, l.stage0);
            CK(cudaMemcpyAsync(pe, l.stage0, sizeof(double) * (size_t)p.nv, cudaMemcpyDeviceToHost, stream));
            CK(cudaStreamSynchronize(stream));
        }
        if (step) *step = step_no;
        CK(cudaGetLastError());
        return MD_OK;
    }

    int pair_tests(long long* tests) override
    {
        if (!tests) { err = "tests is NULL"; return MD_ERR_INVALID_ARG; }
        if (algo == MD_FORCE_ALLPAIRS) {
            *tests = (long long)p.nv * ((long long)p.nv - 1 + p.nw);
            if (dot) {   // the kernel also tests this step's periodic ghost entries
                int g = 0;
                CK(cudaMemcpyAsync(&g, l.ghost_count + gpar, sizeof(int), cudaMemcpyDeviceToHost, stream));
                CK(cudaStreamSynchronize(stream));
                *tests = (long long)p.nv * ((long long)p.nv - 1 + g + (sizeof(T) == 8 ? ad.nwg : adf.nwg));
            }
            return MD_OK;
        }
        if (verlet()) {   // one test per neighbour-list entry
            int rc = refresh();
            if (rc) return rc;
            std::vector<int> h((size_t)p.nv);
            CK(cudaMemcpyAsync(h.data(), l.ncnt, sizeof(int) * h.size(), cudaMemcpyDeviceToHost, stream));
            CK(cudaStreamSynchronize(stream));
            long long t = 0;
            for (int c : h) t += (c & md::VL_NVV_MASK) + ((c >> md::VL_NVW_SHIFT) & md::VL_NVW_MASK);
            *tests = t;
            return MD_OK;
        }
        CK(cudaMemsetAsync(l.tests, 0, sizeof(unsigned long long), stream));
        launch_force<false, false, true>();
        unsigned long long h = 0;
        CK(cudaMemcpyAsync(&h, l.tests, sizeof(h), cudaMemcpyDeviceToHost, stream));
        CK(cudaStreamSynchronize(stream));
        *tests = (long long)h;
        return MD_OK;
    }

    bool pore_region(md::PoreRegion& g) const
    {
        g = md::PoreRegion{};
        if (pore.kind == MD_PORE_SLIT && dim == 2 && (pore.axis == 0 || pore.axis == 1)) g.kind = 1;
        else if (pore.kind == MD_PORE_CYLINDER && dim == 3 && pore.axis >= 0 && pore.axis < 3) g.kind = 2;
        g.axis = pore.axis;
        for (int k = 0; k < 3; ++k) g.c[k] = pore.center[k];
        g.half_len = 0.5 * pore.length; g.r0sq = pore.r0 * pore.r0; g.half_width = 0.5 * pore.width;
        return g.kind != 0;
    }

    int density(int n_axial, long long* axial, int n_radial, double r_max, long long* radial) override
    {
        if (n_axial < 0 || n_radial < 0 || n_axial + n_radial > md::HIST_MAX_BINS || (n_radial > 0 && !(r_max > 0)) ||
            (n_axial > 0 && !axial) || (n_radial > 0 && !radial)) { err = "bad histogram arguments"; return MD_ERR_INVALID_ARG; }
        md::PoreRegion g;
        if (!pore_region(g)) { err = "no monitored pore region (MD_PORE_SLIT in 2D or MD_PORE_CYLINDER in 3D)"; return MD_ERR_UNSUPPORTED; }
        int rc = check_err_flag();
        if (rc) return rc;
        const int nb = n_axial + n_radial;
        if (nb == 0) return MD_OK;
        // profiles run along the pore: the cylinder axis, or (2D slit) the dimension the slit extends in
        const int along = g.kind == 2 ? g.axis : 1 - g.axis;
        unsigned long long* d_out = l.hist;
        CK(cudaMemsetAsync(d_out, 0, sizeof(unsigned long long) * nb, stream));
        md::k_density_profile<T><<<std::min(blocks(256), 296), 256, 0, stream>>>(p, view(), g, along, box.len[along], n_axial,
                                                                              n_radial, r_max > 0 ? r_max : 1.0, d_out);
        std::vector<unsigned long long> h((size_t)nb);
        CK(cudaMemcpyAsync(h.data(), d_out, sizeof(unsigned long long) * nb, cudaMemcpyDeviceToHost, stream));
        CK(cudaStreamSynchronize(stream));
        CK(cudaGetLastError());
        for (int k = 0; k < n_axial; ++k) axial[k] = (long long)h[k];
        for (int k = 0; k < n_radial; ++k) radial[k] = (long long)h[n_axial + k];
        return MD_OK;
    }

    int pressure(md_pressure_out* out) override
    {
        if (!out) { err = "out is NULL"; return MD_ERR_INVALID_ARG; }
        int rc = check_err_flag();
        if (rc) return rc;
        if ((rc = energy_pass())) return rc;               // per-particle virial of the current step
        md::PoreRegion g = {};
        double vol_pore = 0.0;
        const double PI = 3.14159265358979323846;
        if (pore.kind == MD_PORE_SLIT && dim == 2 && (pore.axis == 0 || pore.axis == 1)) {
            g.kind = 1; vol_pore = pore.width * pore.length;
        } else if (pore.kind == MD_PORE_CYLINDER && dim == 3 && pore.axis >= 0 && pore.axis < 3) {
            g.kind = 2; vol_pore = PI * pore.r0 * pore.r0 * pore.length;
        }
        g.axis = pore.axis;
        for (int k = 0; k < 3; ++k) g.c[k] = pore.center[k];
        g.half_len = 0.5 * pore.length; g.r0sq = pore.r0 * pore.r0; g.half_width = 0.5 * pore.width;
        md::k_pressure_partial<T><<<l.red_blocks, md::RED_THREADS, 0, stream>>>(p, view(), l.eo.vir, g, l.part);
        md::k_energy_final<<<1, md::RED_THREADS, 0, stream>>>(l.red_blocks, l.part, l.eout);
        double h[6];
        CK(cudaMemcpyAsync(h, l.eout, sizeof(h), cudaMemcpyDeviceToHost, stream));
        CK(cudaStreamSynchronize(stream));
        CK(cudaGetLastError());
        double vol_box = 1.0;
        for (int k = 0; k < dim; ++k) vol_box *= box.len[k];
        out->volume_box = vol_box;
        out->pressure_box = (2.0 * h[0] + h[1]) / (dim * vol_box);
        out->volume_pore = vol_pore;
        out->kinetic_pore = h[2]; out->virial_pore = h[3]; out->n_pore = (long long)llround(h[4]);
        out->pressure_pore = vol_pore > 0 ? (2.0 * h[2] + h[3]) / (dim * vol_pore) : 0.0;
        out->step = step_no;
        if (g.kind == 0) { err = "no monitored pore region (MD_PORE_SLIT in 2D or MD_PORE_CYLINDER in 3D)"; return MD_ERR_UNSUPPORTED; }
        return MD_OK;
    }

    void info(int* a, int nc[3], int* kps) const override
    {
        if (a) *a = algo;
        if (nc) for (int k = 0; k < 3; ++k) nc[k] = p.nc[k];
        if (kps) *kps = verlet() ? 1 : (algo == MD_FORCE_CELLS ? 5 : (dot ? 3 : 2)) + (p.thermo_rate > 0.0 ? 2 : 0);
    }

    int init(const md_box& box, const md_lj& lj, const md_opts& o, long long nv, const double* pos, const double* vel,
             long long nw, const double* wall);
};

} // namespace

namespace {

template <typename T>
__global__ void k_scatter_wall(int n, const md::Vec4<T>* src, md::Vec4<T>* dst, const int* cell, const int* slot,
                               const int* start)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    dst[start[cell[i]] + slot[i]] = src[i];
}

template <typename T>
int Sim<T>::init(const md_box& box, const md_lj& lj, const md_opts& o, long long nv, const double* pos,
                 const double* vel, long long nw, const double* wall)
{
    // wall particles: upload, convert, and (cell mode) bin once -- they are never integrated
    if (nw > 0) {
        CK(cudaMemcpyAsync(l.wstage, wall, sizeof(double) * (size_t)nw * dim, cudaMemcpyHostToDevice, stream));
        md::State<T> ws = {l.wtr, nullptr, nullptr, nullptr, nullptr};
        md::k_import<T><<<cdiv(nw, 256), 256, 0, stream>>>((int)nw, dim, l.wstage, nullptr, ws);
    }
    CK(cudaMemsetAsync(l.err, 0, 4 * sizeof(int), stream));
    if (algo != MD_FORCE_ALLPAIRS) {
        CK(cudaMemsetAsync(l.count, 0, sizeof(int) * (size_t)p.ncell, stream));
        md::Params<T> pw = p;
        pw.nv = (int)nw;
        if (nw > 0) {
            md::State<T> ws = {l.wtr, nullptr, nullptr, nullptr, nullptr};
            md::k_kick_drift_bin<T, false, true><<<cdiv(nw, 256), 256, 0, stream>>>(pw, ws, l.f, l.count, l.wcell,
                                                                                    l.wslot, l.err);
        }
        launch_scan(l.count, l.wstart);
        if (nw > 0)
            k_scatter_wall<T><<<cdiv(nw, 256), 256, 0, stream>>>((int)nw, l.wtr, l.wr, l.wcell, l.wslot, l.wstart);
        md::k_wall_near<T><<<cdiv(p.ncell, 256), 256, 0, stream>>>(p, l.wstart, l.wnear);
    }
    walls.r = l.wr; walls.start = l.wstart; walls.near = l.wnear;
    // vapor: upload, AoS -> SoA
    CK(cudaMemcpyAsync(l.stage0, pos, sizeof(double) * (size_t)nv * dim, cudaMemcpyHostToDevice, stream));
    CK(cudaMemcpyAsync(l.stage1, vel, sizeof(double) * (size_t)nv * dim, cudaMemcpyHostToDevice, stream));
    md::k_import<T><<<blocks(256), 256, 0, stream>>>((int)nv, dim, l.stage0, l.stage1, l.st[0]);
    cur = 0;
    if (verlet()) {
        // walls (cell order) appended to both position buffers; then bin + list + f(0) in one persistent launch
        CK(cudaMemsetAsync(l.vflags, 0, sizeof(int) * md::VF_COUNT, stream));
        CK(cudaMemsetAsync(l.vtimes, 0, (16 + 8192) * sizeof(unsigned long long), stream));
        CK(cudaMemsetAsync(l.tile_agg, 0, sizeof(unsigned long long) * (size_t)(cdiv(p.ncell, md::SCAN_TILE) + 1), stream));
        if (nw > 0)
            for (int b = 0; b < 2; ++b)
                CK(cudaMemcpyAsync(l.st[b].r + nv, l.wr, sizeof(md::Vec4<T>) * (size_t)nw, cudaMemcpyDeviceToDevice,
                                   stream));
        if constexpr (sizeof(T) == 8)
            if (nw > 0) md::k_wall_ghosts<T><<<cdiv(nw, 256), 256, 0, stream>>>(p, vl);   // fp32 shadow + static ghost copies
        int rc = launch_run(0, 1);
        if (rc) return rc;
        return refresh();
    }
    if (algo == MD_FORCE_CELLS) {
        md::k_kick_drift_bin<T, false, true><<<blocks(256), 256, 0, stream>>>(p, l.st[0], l.f, l.count, l.cell, l.slot,
                                                                             l.err);
        launch_scan(l.count, l.start);
        md::k_scatter<T><<<blocks(256), 256, 0, stream>>>(p.nv, l.st[0], l.st[1], l.f, l.f, l.cell, l.slot, l.start, 0);
        cur = 1;
    }
    if (dot) {
        {
            CK(cudaMemsetAsync(l.ghost_count, 0, 4 * sizeof(int), stream));
            if (nw > 0) {
                if constexpr (std::is_same<T, double>::value)
                    md::k_ap_wall_list<<<cdiv(nw, 256), 256, 0, stream>>>(p, l.wtr, ad, l.ghost_count + 2);
                else
                    md::k_apf_wall_list<<<cdiv(nw, 256), 256, 0, stream>>>(p, adf, l.ghost_count + 2);
            }
            int wg = 0;
            CK(cudaMemcpyAsync(&wg, l.ghost_count + 2, sizeof(int), cudaMemcpyDeviceToHost, stream));
            CK(cudaStreamSynchronize(stream));
            ad.nwg = adf.nwg = (int)nw + wg;
            const int tiles = cdiv(nv, md::AD_THREADS) + cdiv(ad.nwg, md::AD_THREADS) + 1;
            // j slices: enough blocks to fill the GPU, a block count that wastes little of the last wave, and among equals
            // the finer split (measured at N = 65,536: 52 slices 0.625 of the FP64 peak, 128-220 slices 0.631-0.633)
            int dev = 0, sms = 148, nb = 4;
            cudaGetDevice(&dev);
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            ad_ib = nv < md::AD_SMALL_N ? 1 : md::AD_IB;
            if constexpr (std::is_same<T, double>::value)
                cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, md::k_force_allpairs_dot<false, md::AD_IB>, md::AD_THREADS, 0);
            else
                cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, md::k_force_allpairs_dotf<false, md::AD_IB>, md::AD_THREADS, 0);
            const int slots = std::max(1, nb * sms), ib = cdiv(nv, md::AD_THREADS * ad_ib);
            double best = -1.0;
            for (int sl = 1; sl <= std::min(std::max(tiles / 3, 1), 192); ++sl) {
                const double waves = (double)ib * sl / slots;
                const double eff = waves / std::ceil(waves) + (sl * 2e-4) + (waves >= 1.0 ? 0.0 : waves - 1.0);
                if (eff > best) { best = eff; ad_slices = sl; }
            }
            if constexpr (std::is_same<T, double>::value)
                md::k_ap_kick_drift_list<false><<<blocks(256), 256, 0, stream>>>(p, l.st[0], l.f, ad, l.err);
            else
                md::k_apf_kick_drift_list<false><<<blocks(256), 256, 0, stream>>>(p, l.st[0], l.f, adf, l.err);
        }
    }
    launch_force<false, false, false>();   // f(0)
    CK(cudaStreamSynchronize(stream));
    CK(cudaGetLastError());
    return MD_OK;
}

template <typename T>
int create_t(md_sim** out, const md_box& box, const md_pore* pore, const md_lj& lj, const md_opts& o, long long nv, const double* pos,
             const double* vel, long long nw, const double* wall, void* ws, size_t ws_bytes, void* stream,
             const GridSpec& g, int algo)
{
    Sim<T>* s = new Sim<T>();
    const bool cells = algo != MD_FORCE_ALLPAIRS;
    s->dim = box.dim;
    s->box = box;
    s->algo = algo;
    s->stream = (cudaStream_t)stream;
    const int nprune = algo == MD_FORCE_VERLET ? resolve_prunes(box, lj, o) : 0;
    s->l = carve<T>(ws, box.dim, nv, nw, g.ncell, algo, image_blocks(box, o.precision), nprune);
    if (s->l.bytes > ws_bytes) {
        g_create_error = "workspace too small";
        delete s;
        return MD_ERR_WORKSPACE;
    }
    md::Params<T>& p = s->p;
    p.nv = (int)nv; p.nw = (int)nw;
    p.ncell = cells ? (int)g.ncell : 1;
    for (int a = 0; a < 3; ++a) {
        const bool on = a < box.dim;
        p.L[a] = on ? (T)box.len[a] : T(1);
        p.invL[a] = on ? (T)(1.0 / box.len[a]) : T(1);
        p.bc[a] = on ? box.bc[a] : md::BC_NONE;
        p.nc[a] = cells ? g.nc[a] : 1;
        p.inv_c[a] = on ? (T)((double)g.nc[a] / box.len[a]) : T(1);
    }
    auto ucut = [&](double eps, double sig) {
        double q = (sig * sig) / (lj.r_cut * lj.r_cut), q3 = q * q * q;
        return lj.shift_energy ? 4.0 * eps * (q3 * q3 - q3) : 0.0;
    };
    p.rc2 = (T)(lj.r_cut * lj.r_cut);
    p.sig2_vv = (T)(lj.sigma * lj.sigma); p.e24_vv = (T)(24.0 * lj.eps); p.e4_vv = (T)(4.0 * lj.eps);
    p.uc_vv = (T)ucut(lj.eps, lj.sigma);
    p.sig2_vw = (T)(lj.sigma_w * lj.sigma_w); p.e24_vw = (T)(24.0 * lj.eps_w); p.e4_vw = (T)(4.0 * lj.eps_w);
    p.uc_vw = (T)ucut(lj.eps_w, lj.sigma_w);
    p.c12_vv = (T)(48.0 * lj.eps * pow(lj.sigma, 12)); p.c6_vv = (T)(24.0 * lj.eps * pow(lj.sigma, 6));
    p.c12_vw = (T)(48.0 * lj.eps_w * pow(lj.sigma_w, 12)); p.c6_vw = (T)(24.0 * lj.eps_w * pow(lj.sigma_w, 6));
    p.dt = (T)o.dt; p.hk = (T)(o.dt / (2.0 * o.mass)); p.mass = o.mass;
    p.prism = pore && pore->kind == MD_PORE_PRISM;
    p.prism_axis = p.prism ? pore->axis : 0;
    for (int a = 0; a < 3; ++a) {
        const bool on = p.prism && a < box.dim;
        p.prism_c[a] = on ? (T)pore->center[a] : T(0);
        p.prism_h[a] = on ? (T)(0.5 * (a == pore->axis ? pore->length : pore->width)) : T(1);
    }
    p.thermo_rate = o.tau_b > 0 ? o.dt / o.tau_b : 0.0; p.t_target = o.t_target; p.dof = (double)box.dim * (double)nv;
    if (algo == MD_FORCE_ALLPAIRS) {
        // dot-product kernel: needs at most one periodic image per dimension inside r_c + margin of a face
        bool ok = true;
        for (int a = 0; a < box.dim; ++a)
            if (box.bc[a] == MD_BC_PERIODIC && box.len[a] < 2.2 * lj.r_cut) ok = false;
        if (ok) {
            md::AllPairsDot& a = s->ad;
            s->dot = true;
            if constexpr (std::is_same<T, double>::value) { a.jv = s->l.jv; a.jw = s->l.jw; }
            a.ghost_count = s->l.ghost_count; a.nwg = 0;
            // Origin: x' = x + shift with shift^2 > thr makes |r_i|^2 - thr > 0 for every particle in the box (the filter
            // compares positive numbers through their bits, md_allpairs.cuh); y, z: box centre.  thr = r_c^2 plus a bound
            // on the rounding of the dot-product form and of |r_i|^2 - thr, which grows with the largest |coordinate| of
            // an entry (ghosts included) and so with the shift itself: r_c + 1 unless the box is thousands of sigma wide
            // in fp32 mode (~6 eps32 |r|^2 terms; fp64: 64 x 2.3e-16 |r|^2).
            constexpr bool F32 = std::is_same<T, float>::value;
            double shift = lj.r_cut + 1.0, thr = 0.0;
            for (int it = 0; it < 8; ++it) {
                double smax = 0.0;
                for (int k = 0; k < box.dim; ++k) {
                    const double h = (k == 0 ? box.len[k] + shift : 0.5 * box.len[k]) + 1.1 * lj.r_cut;
                    smax += 2.0 * h * h;
                }
                thr = lj.r_cut * lj.r_cut + (F32 ? 1e-6 * smax + 1e-3 : 64.0 * 2.3e-16 * smax + 1e-12);
                if (shift * shift > 1.05 * thr) break;
                shift = std::sqrt(1.05 * thr) + 1.0;
            }
            for (int k = 0; k < 3; ++k) a.org[k] = k < box.dim ? 0.5 * box.len[k] : 0.0;
            a.org[0] = -shift;
            a.edge = lj.r_cut * (1.0 + 1e-9) + 1e-9;
            a.thr = thr;
            if constexpr (F32) {
                md::AllPairsDotF& g = s->adf;
                g.jv = s->l.jv; g.jw = s->l.jw; g.jv_id = s->l.jv_id; g.jw_id = s->l.jw_id; g.wr = s->l.wtr;
                g.ghost_count = s->l.ghost_count; g.nwg = 0;
                for (int k = 0; k < 3; ++k) g.org[k] = (float)a.org[k];
                g.edge = (float)(lj.r_cut * (1.0 + 1e-5) + 1e-4);
                g.thr = (float)thr;
            }
        }
    }
    if (algo == MD_FORCE_VERLET) {
        const double skin = list_skin(lj, o), rl = lj.r_cut + skin;
        md::Verlet<T>& v = s->vl;
        v.st[0] = s->l.st[0]; v.st[1] = s->l.st[1]; v.f = s->l.f;
        v.nbr = s->l.nbr; v.ncnt = s->l.ncnt;      // lists: warp-blocked, n = align_up(nv, 64) particles allocated
        v.cell = s->l.cell; v.slot = s->l.slot; v.count = s->l.count; v.start = s->l.start; v.tile_agg = s->l.tile_agg;
        v.wstart = s->l.wstart; v.wnear = s->l.wnear; v.flags = s->l.vflags; v.bar = s->l.vbar; v.ksum = s->l.vksum; v.times = s->l.vtimes;
        v.dbg = nullptr;
        v.r32 = s->l.r32;
        v.onbr = s->l.onbr; v.ocnt = s->l.ocnt; v.oheavy = s->l.oheavy; v.wo = s->l.wo;
        v.nprune = nprune;
        const double so = outer_skin(skin, nprune), rlo = lj.r_cut + so;
        v.outer_lim = (T)(0.5 * (so - skin));
        v.ntot = (int)(nv + nw); v.nimg = image_blocks(box, o.precision);
        v.half_skin = (T)(0.5 * skin);
        // fp32 filter of the list build: (r_c + skin) plus the rounding of the fp32 positions (ulp(L) / 2 each), of the
        // image shift (ulp(2L) / 2) and of the fma chain; the list only has to be a superset
        double lmax = 0.0;
        for (int a = 0; a < box.dim; ++a) lmax = std::max(lmax, box.len[a]);
        const double rlf = rl * (1.0 + 4e-7) + 4.0 * lmax * 1.1920929e-7;
        v.rl2f = (float)(rlf * rlf * (1.0 + 2e-7));
        const double rlof = rlo * (1.0 + 4e-7) + 4.0 * lmax * 1.1920929e-7;
        v.rl2f_out = (float)(rlof * rlof * (1.0 + 2e-7));
        // the prune tests the positions themselves: exact threshold in fp64 (plus 1e-9: the path lengths are rounded up
        // by 1e-6, see step_len), the build's inflated one in fp32
        v.rl2_prune = sizeof(T) == 8 ? (T)(rl * rl * (1.0 + 1e-9)) : (T)v.rl2f;
        v.heavy_t = o.heavy_list > 0 ? o.heavy_list - 1 : 12;   // lists of heavy_list entries or more (default 13)
        v.carry = 1;
#ifdef MD_DIAGNOSTICS
        if (getenv("MD_DEBUG_TIMES")) v.dbg = s->l.vtimes + 16;
        if (getenv("MD_NO_CARRY")) v.carry = 0;
#endif
    }
    int rc = s->init(box, lj, o, nv, pos, vel, nw, wall);
    if (rc != MD_OK) {
        g_create_error = s->err;
        delete s;
        return rc;
    }
    *out = s;
    return MD_OK;
}

template <typename T>
double time_fma(cudaStream_t st, T* out, cudaEvent_t a, cudaEvent_t b)
{
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int grid = sms * 8, iters = 1 << 14;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(a, st);
        md::k_fma_chain<T><<<grid, 256, 0, st>>>(iters, T(1), out);
        cudaEventRecord(b, st);
        cudaEventSynchronize(b);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, a, b);
        double tf = 2.0 * 8.0 * iters * 256.0 * grid / (ms * 1e-3) * 1e-12;
        if (rep > 0 && tf > best) best = tf;
    }
    return best;
}

} // namespace

extern "C" {

size_t md_workspace_bytes(const md_box* box, const md_lj* lj, const md_opts* o, long long nv, long long nw)
{
    if (validate(box, lj, o, nv, nw)) return 0;
    int algo = pick_algo(*box, *lj, *o, nv, nw);
    if (algo < 0) return 0;
    GridSpec g = grid_for(*box, *lj, *o, algo);
    const int nimg = image_blocks(*box, o->precision), nprune = algo == MD_FORCE_VERLET ? resolve_prunes(*box, *lj, *o) : 0;
    return o->precision == 64 ? carve<double>(nullptr, box->dim, nv, nw, g.ncell, algo, nimg, nprune).bytes
                              : carve<float>(nullptr, box->dim, nv, nw, g.ncell, algo, nimg, nprune).bytes;
}

int md_create(md_sim** out, const md_box* box, const md_pore* pore, const md_lj* lj, const md_opts* o, long long nv,
              const double* pos, const double* vel, long long nw, const double* wall, void* ws, size_t ws_bytes,
              void* stream)
{
    if (!out) { g_create_error = "out is NULL"; return MD_ERR_INVALID_ARG; }
    *out = nullptr;
    const char* why = validate(box, lj, o, nv, nw);
    if (!why && (!pos || !vel)) why = "pos / vel is NULL";
    if (!why && nw > 0 && !wall) why = "wall_pos is NULL with n_wall > 0";
    if (!why && (!ws || ((uintptr_t)ws & 255))) why = "device_workspace is NULL or not 256-byte aligned";
    if (why) { g_create_error = why; return MD_ERR_INVALID_ARG; }
    const int dim = box->dim;
    auto inside = [&](const double* r, long long n) {
        for (long long i = 0; i < n; ++i)
            for (int a = 0; a < dim; ++a) {
                double v = r[i * dim + a];
                if (!(v >= 0.0 && v <= box->len[a])) return false;   // also rejects NaN
            }
        return true;
    };
    if (!inside(pos, nv) || !inside(wall, nw)) { g_create_error = "position non-finite or outside [0, L]"; return MD_ERR_INVALID_ARG; }
    for (long long i = 0; i < nv * dim; ++i)
        if (!std::isfinite(vel[i])) { g_create_error = "velocity non-finite"; return MD_ERR_INVALID_ARG; }
    int algo = pick_algo(*box, *lj, *o, nv, nw);
    if (algo < 0) { g_create_error = "cell list needs >= 3 cells in every periodic dimension"; return MD_ERR_UNSUPPORTED; }
    GridSpec g = grid_for(*box, *lj, *o, algo);
    if (pore && pore->kind == MD_PORE_PRISM) {
        // geometric walls must sit inside the box with a margin (VERLET keeps periodic coordinates unwrapped by < skin)
        if (pore->axis < 0 || pore->axis >= dim || !(pore->length > 0) || !(pore->width > 0)) {
            g_create_error = "prism pore needs 0 <= axis < dim, length > 0, width > 0";
            return MD_ERR_INVALID_ARG;
        }
        for (int a = 0; a < dim; ++a) {
            const double h = 0.5 * (a == pore->axis ? pore->length : pore->width);
            // VERLET leaves periodic coordinates unwrapped between FULL rebuilds: by up to (outer skin - skin) / 2 + skin / 2
            // + one step with the two-level list
            const double margin = std::max(1.0, outer_skin(list_skin(*lj, *o), resolve_prunes(*box, *lj, *o)));
            if (!(pore->center[a] - h >= margin) || !(pore->center[a] + h <= box->len[a] - margin)) {
                g_create_error = "prism pore must lie at least max(1, outer skin) length units inside the box";
                return MD_ERR_INVALID_ARG;
            }
        }
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        g_create_error = "no CUDA device (there is no CPU fallback)";
        return MD_ERR_CUDA;
    }
    int rc = o->precision == 64
                 ? create_t<double>(out, *box, pore, *lj, *o, nv, pos, vel, nw, wall, ws, ws_bytes, stream, g, algo)
                 : create_t<float>(out, *box, pore, *lj, *o, nv, pos, vel, nw, wall, ws, ws_bytes, stream, g, algo);
    if (rc == MD_OK && pore) (*out)->pore = *pore;
    return rc;
}

int md_step(md_sim* s, long long n) { return s ? s->step(n) : MD_ERR_INVALID_ARG; }
int md_get_state(md_sim* s, double* pos, double* vel, double* force, double* pe, long long* step)
{
    return s ? s->get_state(pos, vel, force, pe, step) : MD_ERR_INVALID_ARG;
}
int md_energy(md_sim* s, md_energy_out* out) { return s ? s->energy(out) : MD_ERR_INVALID_ARG; }
int md_profile_step(md_sim* s, long long n, md_kernel_times* out) { return s ? s->profile(n, out) : MD_ERR_INVALID_ARG; }
int md_pair_tests(md_sim* s, long long* t) { return s ? s->pair_tests(t) : MD_ERR_INVALID_ARG; }
int md_pressure(md_sim* s, md_pressure_out* out) { return s ? s->pressure(out) : MD_ERR_INVALID_ARG; }
int md_density_profile(md_sim* s, int na, long long* axial, int nr, double r_max, long long* radial)
{
    return s ? s->density(na, axial, nr, r_max, radial) : MD_ERR_INVALID_ARG;
}
int md_info(const md_sim* s, int* algo, int nc[3], int* kps)
{
    if (!s) return MD_ERR_INVALID_ARG;
    s->info(algo, nc, kps);
    return MD_OK;
}
int md_destroy(md_sim* s)
{
    if (s) s->drain();          // the workspace is the caller's: nothing of ours may still run on it afterwards
    delete s;
    return MD_OK;
}
const char* md_last_error(const md_sim* s) { return s ? s->err.c_str() : g_create_error.c_str(); }

int md_measure_peaks(void* scratch, size_t bytes, void* stream, md_peaks* out)
{
    if (!scratch || !out || bytes < (1u << 20)) return MD_ERR_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return MD_ERR_CUDA; }
    cudaStream_t st = (cudaStream_t)stream;
    cudaEvent_t a, b;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return MD_ERR_CUDA;
    out->fp64_tflops = time_fma<double>(st, (double*)scratch, a, b);
    out->fp32_tflops = time_fma<float>(st, (float*)scratch, a, b);
    size_t n16 = bytes / 32;   // double2 elements per half
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(a, st);
        md::k_copy<<<148 * 16, 256, 0, st>>>((const double2*)scratch, (double2*)scratch + n16, n16);
        cudaEventRecord(b, st);
        cudaEventSynchronize(b);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, a, b);
        double gbs = 2.0 * 16.0 * (double)n16 / (ms * 1e-3) * 1e-9;
        if (rep > 0 && gbs > best) best = gbs;
    }
    out->copy_gbs = best;
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    return cudaGetLastError() == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

} // extern "C"
