/*
 * md.h -- C ABI of the B200-native Lennard-Jones pore-MD hot path.
 *
 * What it computes (arxiv 1812.07993, Korenkov / Nikonov / Popovicova):
 *   - Newton's equations m_i r''_i = f_i, f_i = -dU/dr_i        PAPER.md:35-43, Eq. (1)-(2)
 *   - U = sum of Lennard-Jones pair terms
 *   - velocity Verlet: F2 (r(t+dt), v(t+dt/2)), F1 (forces from r(t+dt)),
 *     F3 (v(t+dt))                                                 PAPER.md:57, :69-93 (Figs. 1-3)
 *   - periodic / reflecting boundaries
 *   plus, from BASELINE.json's north_star (not in the paper): cut-off r_c, fixed
 *   wall particles (eps_w, sigma_w), cell-list neighbour search, K/U reductions,
 *   optional fp32 mode.  Readings of every silent point: DESIGN.md "Readings".
 *
 * Conventions
 *   Ownership : the caller owns every host array and the device workspace.  The
 *               library never calls cudaMalloc; md_create copies its inputs and
 *               keeps no host pointer.  The workspace must outlive the handle.
 *   Pointers  : "host" = ordinary host memory; "device" = CUDA device memory on
 *               the current device.  All particle arrays at the boundary are
 *               fp64, row-major [n][dim] (AoS), in the caller's ORIGINAL particle
 *               order regardless of internal sorting.
 *   Errors    : every call returns an int status (MD_OK = 0, negatives below); no
 *               exception or abort crosses the boundary; text via md_last_error.
 *   Streams   : md_step only enqueues work on the stream given to md_create;
 *               md_get_state / md_energy / md_profile_step / md_pair_tests
 *               synchronise that stream before returning.
 *   Time      : md_get_state / md_energy report r(t), v(t), f(t) of the same
 *               integer step t.
 *   Threads   : one handle is used by one host thread at a time.
 *   There is no CPU fallback: without a CUDA device every compute call fails
 *   with MD_ERR_CUDA.
 */
#ifndef PAPER_1812_07993_MD_H
#define PAPER_1812_07993_MD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct md_sim md_sim; /* opaque */

enum { MD_OK = 0, MD_ERR_INVALID_ARG = -1, MD_ERR_UNSUPPORTED = -2, MD_ERR_CUDA = -3,
       MD_ERR_WORKSPACE = -4, MD_ERR_NONFINITE = -5, MD_ERR_STATE = -6 };
enum { MD_BC_PERIODIC = 0, MD_BC_REFLECT = 1 };
enum { MD_FORCE_AUTO = 0, MD_FORCE_ALLPAIRS = 1, MD_FORCE_CELLS = 2, MD_FORCE_VERLET = 3 };
enum { MD_PORE_NONE = 0, MD_PORE_SLIT, MD_PORE_CYLINDER, MD_PORE_CONE, MD_PORE_INKBOTTLE, MD_PORE_PRISM };

/* Simulation box [0, len[d]] per dimension; dim = 2 or 3 (len[2], bc[2] ignored in 2D).
 * bc[d]: MD_BC_PERIODIC (positions kept in [0, len), nearest image) or
 * MD_BC_REFLECT (specular reflection after the drift). */
typedef struct { int dim; double len[3]; int bc[3]; } md_box;

/* Pore region.  The hot path sees wall PARTICLES, not shapes; the descriptor only selects the volume md_pressure
 * monitors: MD_PORE_CYLINDER (3D): distance from the axis line through `center` along dimension `axis` < r0 and
 * |along - center[axis]| < length/2; MD_PORE_SLIT (2D): |r[axis] - center[axis]| < width/2 (axis = wall normal) and
 * |r[1-axis] - center[1-axis]| < length/2.  MD_PORE_PRISM switches on GEOMETRIC walls (the paper's own pore,
 * PAPER.md:115-121, :186): the axis-aligned box of size `length` along `axis` and `width` across, centred at `center`,
 * reflects particles specularly from both sides of every face except the open one at +axis; it must lie at least
 * max(1, outer skin) length units inside the simulation box (outer skin: see md_opts.list_prunes; 1.93 by default).  Other kinds are stored but neither monitored nor active. */
typedef struct { int kind, axis; double center[3], length, r0, r1, neck_len, width; } md_pore;

/* 12-6 Lennard-Jones: u(r) = 4 eps [(sigma/r)^12 - (sigma/r)^6] for r < r_cut, else 0 (strict <);
 * vapor-vapor (eps, sigma), vapor-wall (eps_w, sigma_w), same r_cut.  shift_energy != 0 subtracts
 * u(r_cut) inside the cut-off (energies only; the force is plainly truncated). */
typedef struct { double eps, sigma, eps_w, sigma_w, r_cut; int shift_energy; } md_lj;

/* dt > 0, mass > 0 (one mass for all vapor particles); precision 64 or 32 (state and pair
 * arithmetic type; K and U are always reduced in fp64); force_algo one of MD_FORCE_*:
 *   ALLPAIRS  shared-memory-tiled all-pairs (small N);
 *   CELLS     counting-sort cell list rebuilt every step, neighbour-cell traversal;
 *   VERLET    the same cell list, rebuilt only when a particle's path since the last rebuild exceeds
 *             skin/2, cached as a neighbour list of all pairs within r_cut + skin (exact: no pair
 *             within r_cut is ever missed); the whole md_step batch is one persistent launch;
 *   AUTO      VERLET when the box holds >= 3 cells of side r_cut + skin per periodic dimension, else CELLS
 *             under the same rule with r_cut, else ALLPAIRS.
 * 0 <= skin < r_cut is the VERLET list margin in length units; 0 selects the default 0.24 r_cut.
 * heavy_list >= 0: VERLET lists of this many entries or more are walked by a group of four lanes instead of the
 * particle's own thread (0 selects the default 13; a tuning knob, results do not depend on it).
 * list_prunes: VERLET two-level list: between two full rebuilds (bin, scan, scatter, cell walk) the r_cut + skin list is
 * pruned that many times from an outer list of all pairs within r_cut + outer skin, outer skin = 1.07 (list_prunes + 1)
 * skin; 0 selects the default 2, < 0 none (single-level list), at most 8; reduced automatically while the box does not hold
 * 3 cells of side r_cut + outer skin per periodic dimension.  Exact either way: a prune that finds a particle whose path
 * since the full rebuild exceeds (outer skin - skin) / 2 is discarded and a full rebuild runs instead.
 * tau_b > 0 switches on the Berendsen thermostat (the paper's kernel F4) after every step:
 * v <- lambda v, lambda = sqrt(1 + (dt / tau_b)(t_target / T - 1)), T = 2K / (dim n_vapor) (k_B = 1); tau_b <= 0: NVE. */
typedef struct { double dt, mass; int precision, force_algo; double skin; double tau_b, t_target; int heavy_list, list_prunes; } md_opts;

/* potential = potential_vv + potential_vw = sum_i pe_i; virial = sum over unordered vv pairs and
 * vw pairs of g.d (g = force on the vapor particle, d = r_i - r_j); pairs_* = pairs with r < r_cut. */
typedef struct { double kinetic, potential, potential_vv, potential_vw, virial;
                 long long pairs_vv, pairs_vw; long long step; } md_energy_out;

/* Virial pressure: P = (2K + W) / (dim V), K and W = sum_i (1/2 sum_j g.d + sum_w g.d) summed over
 * the particles inside the volume (k_B = 1; W as in md_energy_out.virial: positive = repulsive.  The paper prints the
 * virial term with a minus sign, i.e. with the opposite sign convention for f(r_ij): DESIGN.md reading A17). */
typedef struct { double pressure_box, volume_box, pressure_pore, volume_pore, kinetic_pore, virial_pore;
                 long long n_pore; long long step; } md_pressure_out;

/* Per-kernel device times of md_profile_step, milliseconds summed over the profiled steps, and
 * launch counts.  Index: 0 kick+drift(+bin count), 1 scan, 2 scatter, 3 force(+half-kick).  VERLET: the
 * whole batch is one launch, reported in slot 3 (slots 0-2: step phases, grid barriers, rebuilds as timed inside the
 * kernel by its first thread); rebuilds = cell-list + neighbour-list rebuilds in it, rebuild_ms = their split into
 * bin, scan, scatter and list build, each with the grid barrier that ends it; prunes = list prunes in it (two-level list),
 * prune_ms their time, also counted in ms[2] (VERLET only, else 0). */
typedef struct { double ms[4]; long long launches[4]; double total_ms; long long steps, rebuilds; double rebuild_ms[4];
                 long long prunes; double prune_ms; } md_kernel_times;

/* Peak micro-benchmarks run on the caller's stream (TFLOP/s count FMA = 2 flops; GB/s = read+write). */
typedef struct { double fp64_tflops, fp32_tflops, copy_gbs; } md_peaks;

/* Bytes of device workspace md_create needs for these arguments (0 on invalid arguments). */
size_t md_workspace_bytes(const md_box*, const md_lj*, const md_opts*, long long n_vapor, long long n_wall);

/* Builds a simulation: validates, uploads pos/vel (host [n_vapor][dim]) and wall_pos (host
 * [n_wall][dim], may be NULL iff n_wall == 0), bins, evaluates f(0).  device_workspace: device
 * memory of >= md_workspace_bytes bytes, 256-byte aligned.  cuda_stream: a cudaStream_t (NULL =
 * default stream).  pore may be NULL.  Invalid: dim not 2/3, n_vapor < 1, n_wall < 0, dt <= 0,
 * mass <= 0, r_cut <= 0, non-finite or out-of-box positions, a periodic length < 2 r_cut, skin < 0 or >= r_cut, a thermostat
 * with tau_b < dt or t_target <= 0, a prism pore not inside the box.
 * MD_ERR_UNSUPPORTED: MD_FORCE_CELLS with a periodic dimension shorter than 3 cells (AUTO falls
 * back to all-pairs).  On failure *out = NULL and md_last_error(NULL) has the reason. */
int md_create(md_sim** out, const md_box*, const md_pore*, const md_lj*, const md_opts*,
              long long n_vapor, const double* pos, const double* vel,
              long long n_wall, const double* wall_pos,
              void* device_workspace, size_t workspace_bytes, void* cuda_stream);

/* Enqueues n_steps velocity-Verlet steps (F2 -> [re-bin] -> F1 -> F3 per step). Asynchronous. */
int md_step(md_sim*, long long n_steps);

/* Copies the state at the current step to host buffers (each may be NULL = skip):
 * pos, vel, force [n_vapor][dim]; pe [n_vapor] (pe_i = 1/2 sum_j u_vv + sum_w u_vw); *step.
 * MD_ERR_STATE if a particle left a reflecting box (more than one bounce in a step);
 * MD_ERR_WORKSPACE if a VERLET neighbour list overflowed its 128 entries per particle. */
int md_get_state(md_sim*, double* pos, double* vel, double* force, double* pe, long long* step);

/* Kinetic / potential energies, virial and pair counts at the current step (host struct).
 * MD_ERR_NONFINITE if K or U is not finite. */
int md_energy(md_sim*, md_energy_out* out);

/* Box pressure and pressure inside the pore region given to md_create at the current step (host struct).
 * MD_ERR_UNSUPPORTED if no monitored pore kind was given (pressure_box is still filled). */
int md_pressure(md_sim*, md_pressure_out* out);

/* Vapor density profiles about the pore given to md_create, histogrammed on the device at the current step
 * (NEXT-4; the long-run comparison of north_star).  axial[n_axial]: particle counts in equal slabs of the whole box
 * length along pore.axis.  radial[n_radial]: counts in equal-width shells 0 <= rho < r_max about the axis line through
 * pore.center, restricted to |along - center| < length/2 (3D cylinder; in 2D rho = |r[axis] - center[axis]| with axis
 * the wall normal and the restriction along the other dimension).  Host int64 arrays, either may be NULL.
 * MD_ERR_UNSUPPORTED without a monitored pore kind. */
int md_density_profile(md_sim*, int n_axial, long long* axial, int n_radial, double r_max, long long* radial);

/* Like md_step but synchronous, one launch at a time with CUDA events around every kernel. */
int md_profile_step(md_sim*, long long n_steps, md_kernel_times* out);

/* Ordered candidate distance tests one force evaluation performs at the current state
 * (vapor-vapor + vapor-wall), counted by an untimed instrumented pass. */
int md_pair_tests(md_sim*, long long* tests);

/* Which force path the handle uses (MD_FORCE_ALLPAIRS / MD_FORCE_CELLS / MD_FORCE_VERLET), its cell grid, and the
 * kernels launched per time step (VERLET: 1 = the whole md_step batch is one persistent launch). */
int md_info(const md_sim*, int* force_algo, int n_cells[3], int* kernels_per_step);

/* DFMA / FFMA chains on every SM and a device copy; scratch = device memory, >= 64 MiB for a
 * meaningful copy figure. */
int md_measure_peaks(void* device_scratch, size_t scratch_bytes, void* cuda_stream, md_peaks* out);

/* Kinetic energy K = sum_i 1/2 m |v_i|^2 (row a5; the quantity the thermostat F4 needs every step, PAPER.md:45, :94-102,
 * :111) for callers that cannot allocate device memory: code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc.  Needs no handle and no workspace: the per-block partial sums of the reduction live in a static
 * __device__ array inside the library (32 KiB on every GPU that loads it, until the process exits), which is why n is
 * limited to MD_NOALLOC_MAX_PARTICLES.  vel_device: DEVICE memory, fp64 [n][dim] (row-major, as at md_create's boundary);
 * kinetic_device: DEVICE memory, one double, written by the call; both stay the caller's.  Asynchronous on cuda_stream
 * (NULL = default stream); the first call on a device resolves the array's address (set-up), later calls only launch two
 * kernels.  Calls no cudaMalloc / cudaFree / allocating routine.  All calls share the one scratch array: calls that overlap
 * on the GPU (different streams or host threads) race on it -- serialise them; nothing needs clearing between calls.
 * errbuf (host, may be NULL) receives the reason on failure.  MD_ERR_INVALID_ARG: NULL pointers, dim not 2/3, mass <= 0,
 * n < 1; MD_ERR_WORKSPACE: n > MD_NOALLOC_MAX_PARTICLES; MD_ERR_CUDA: no device, or a CUDA error. */
#define MD_NOALLOC_MAX_PARTICLES 4194304
int md_kinetic_energy_noalloc(const double* vel_device, long long n, int dim, double mass, double* kinetic_device,
                              void* cuda_stream, char* errbuf, size_t errbuf_len);

int md_destroy(md_sim*);
const char* md_last_error(const md_sim*); /* NULL handle: this thread's last md_create error */

#ifdef __cplusplus
}
#endif
#endif
