/*
 * md_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU statement of the hot path of
 * arxiv 1812.07993 (Korenkov, Nikonov, Popovicova): pairwise Lennard-Jones
 * forces (kernel F1, Fig. 1 at :69-73) and the velocity-Verlet
 * update (kernels F2/F3), Newton's equations Eq. (1)-(2)
 * (PAPER.md:35-43), with the cut-off, fixed wall particles and energies that
 * BASELINE.json's north_star adds (readings A1-A7 in DESIGN.md).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load this file's library.  It shares no code, header,
 * table or helper with paper_1812_07993_b200/csrc and neither includes the
 * other.  fp64 throughout; compiled -O2 -ffp-contract=off (only the explicit
 * fma() calls below fuse), OpenMP over the particle loop, no blocking, no
 * vectorisation by hand, no Newton-third-law sharing.
 *
 * Pins (tests/test_oracle_pins.py): two-particle closed form, wall closed
 * form, Newton's third law, translation invariance / minimum image, free
 * flight, bound-pair harmonic period, dt^2 energy-error order, time
 * reversibility, energy conservation, cell list == brute force, scipy pdist
 * sum.  Long chaotic runs (configs 1-4 beyond 100 steps) are "parity
 * unpinned" pointwise and compared statistically only.
 *
 * Layouts: pos, vel, f are host arrays [n][dim] (AoS, as at the product's
 * boundary); pe, pe_w, vir are [n].
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int dim;            /* 2 or 3 */
    double L[3];        /* box lengths */
    int bc[3];          /* 0 periodic, 1 reflecting */
    double eps, sigma;  /* vapor-vapor */
    double eps_w, sigma_w; /* vapor-wall */
    double r_cut;
    int shift_energy;   /* 1: u(r) - u(r_c) inside the cut-off (reading A2) */
    double dt, mass;
    double tau_b, t_target; /* Berendsen thermostat F4: rise time (<= 0: off), T_0 */
    /* NEXT-3, the paper's own pore: an axis-aligned box whose faces reflect from both sides, except the face at
     * +prism_axis, which is open (2D: square pore with three closed sides; 3D: prism with five
     * isolated walls and one open).  prism = 0: none. */
    int prism, prism_axis;
    double prism_c[3], prism_h[3]; /* centre, half sizes */
} orc_params;

/* ---- c.1 definitions ------------------------------------------------- */

/* Minimum image per periodic dimension: d <- d - L*rint(d/L) (reading A3). */
static void min_image(const orc_params *p, double *d)
{
    for (int a = 0; a < p->dim; ++a)
        if (p->bc[a] == 0)
            d[a] = d[a] - p->L[a] * rint(d[a] / p->L[a]);
}

/* r^2 with the fixed FMA order of SURVEY 8(c) c.1 so the strict r^2 < r_c^2
 * decision is taken in the same arithmetic on both sides. */
static double norm2(int dim, const double *d)
{
    double r2 = fma(d[1], d[1], d[0] * d[0]);
    if (dim == 3) r2 = fma(d[2], d[2], r2);
    return r2;
}

/* u_c = 4 eps [(sigma/r_c)^12 - (sigma/r_c)^6] */
static double u_cut(double eps, double sigma, double r_cut)
{
    double s = (sigma * sigma) / (r_cut * r_cut);
    double s3 = s * s * s;
    return 4.0 * eps * (s3 * s3 - s3);
}

/* One ordered pair (i <- j) with displacement d = r_i - r_j (already minimum
 * image).  Standard 12-6 Lennard-Jones (reading A1):
 *   u = 4 eps (s^6 - s^3) - u_c,   g = (24 eps / r^2)(2 s^6 - s^3),  s = sigma^2/r^2
 * Returns 1 if r^2 < r_c^2 (strict), else 0 and leaves outputs untouched. */
static int lj_pair(double eps, double sigma, double rc2, double uc, int dim, const double *d,
                   double *g_over_r2_out, double *u_out, double *r2_out)
{
    double r2 = norm2(dim, d);
    if (!(r2 < rc2)) return 0;
    double s = (sigma * sigma) / r2;
    double s3 = s * s * s;
    double s6 = s3 * s3;
    *u_out = 4.0 * eps * (s6 - s3) - uc;
    *g_over_r2_out = (24.0 * eps / r2) * (2.0 * s6 - s3);
    *r2_out = r2;
    return 1;
}

/* ---- c.2 brute-force forces and energies ----------------------------- */
/* f_i = sum_{j != i} g_vv + sum_w g_vw ; pe_i = 1/2 sum u_vv + sum u_vw ;
 * vir_i = 1/2 sum g.d (vv) + sum g.d (vw) ; pe_w_i = sum u_vw.
 * counts[0] = ordered vapor-vapor hits, counts[1] = vapor-wall hits.
 * j ascending, j == i skipped by index. Any of pe, pe_w, vir, counts may be NULL. */
void orc_forces_brute(const orc_params *p, long nv, const double *pos, long nw, const double *wall,
                      double *f, double *pe, double *pe_w, double *vir, long long *counts)
{
    const int dim = p->dim;
    const double rc2 = p->r_cut * p->r_cut;
    const double uc_vv = p->shift_energy ? u_cut(p->eps, p->sigma, p->r_cut) : 0.0;
    const double uc_vw = p->shift_energy ? u_cut(p->eps_w, p->sigma_w, p->r_cut) : 0.0;
    long long c_vv = 0, c_vw = 0;
#pragma omp parallel for schedule(static) reduction(+ : c_vv, c_vw)
    for (long i = 0; i < nv; ++i) {
        double fi[3] = {0.0, 0.0, 0.0}, u_vv = 0.0, u_vw = 0.0, w_vv = 0.0, w_vw = 0.0;
        for (long j = 0; j < nv; ++j) {
            if (j == i) continue;
            double d[3] = {0.0, 0.0, 0.0}, g, u, r2;
            for (int a = 0; a < dim; ++a) d[a] = pos[i * dim + a] - pos[j * dim + a];
            min_image(p, d);
            if (lj_pair(p->eps, p->sigma, rc2, uc_vv, dim, d, &g, &u, &r2)) {
                for (int a = 0; a < dim; ++a) fi[a] += g * d[a];
                u_vv += u;
                w_vv += g * r2;
                ++c_vv;
            }
        }
        for (long w = 0; w < nw; ++w) {
            double d[3] = {0.0, 0.0, 0.0}, g, u, r2;
            for (int a = 0; a < dim; ++a) d[a] = pos[i * dim + a] - wall[w * dim + a];
            min_image(p, d);
            if (lj_pair(p->eps_w, p->sigma_w, rc2, uc_vw, dim, d, &g, &u, &r2)) {
                for (int a = 0; a < dim; ++a) fi[a] += g * d[a];
                u_vw += u;
                w_vw += g * r2;
                ++c_vw;
            }
        }
        for (int a = 0; a < dim; ++a) f[i * dim + a] = fi[a];
        if (pe) pe[i] = 0.5 * u_vv + u_vw;
        if (pe_w) pe_w[i] = u_vw;
        if (vir) vir[i] = 0.5 * w_vv + w_vw;
    }
    if (counts) { counts[0] = c_vv; counts[1] = c_vw; }
}

/* ---- c.4 CPU cell-list variant (long runs only) ----------------------- */
/* Grid rule (reading A10/A11): n_d = max(1, floor(L_d / r_c)), c_d = L_d / n_d,
 * cell index floor(r_d / c_d) clamped to [0, n_d - 1]; neighbour offsets
 * -1, 0, +1 wrapped in periodic dimensions (needs n_d >= 3), dropped outside
 * the box in reflecting dimensions. */
typedef struct {
    int n[3];
    long ncell;
    long *start;   /* [ncell + 1] */
    long *items;   /* particle indices in cell order (stable by index) */
} orc_grid;

static long cell_of(const orc_params *p, const orc_grid *g, const double *r)
{
    long c[3] = {0, 0, 0};
    for (int a = 0; a < p->dim; ++a) {
        double w = p->L[a] / (double)g->n[a];
        long k = (long)floor(r[a] / w);
        if (k < 0) k = 0;
        if (k > g->n[a] - 1) k = g->n[a] - 1;
        c[a] = k;
    }
    return (c[2] * g->n[1] + c[1]) * g->n[0] + c[0];
}

static int grid_build(const orc_params *p, orc_grid *g, long n, const double *pos)
{
    g->n[0] = g->n[1] = g->n[2] = 1;
    for (int a = 0; a < p->dim; ++a) {
        int k = (int)floor(p->L[a] / p->r_cut);
        if (k < 1) k = 1;
        if (p->bc[a] == 0 && k < 3) return -1;
        g->n[a] = k;
    }
    g->ncell = (long)g->n[0] * g->n[1] * g->n[2];
    g->start = (long *)calloc((size_t)g->ncell + 1, sizeof(long));
    g->items = (long *)malloc(sizeof(long) * (size_t)(n > 0 ? n : 1));
    long *cid = (long *)malloc(sizeof(long) * (size_t)(n > 0 ? n : 1));
    for (long i = 0; i < n; ++i) { cid[i] = cell_of(p, g, pos + i * p->dim); g->start[cid[i] + 1]++; }
    for (long c = 0; c < g->ncell; ++c) g->start[c + 1] += g->start[c];
    long *fill = (long *)malloc(sizeof(long) * (size_t)g->ncell);
    memcpy(fill, g->start, sizeof(long) * (size_t)g->ncell);
    for (long i = 0; i < n; ++i) g->items[fill[cid[i]]++] = i;
    free(fill); free(cid);
    return 0;
}

static void grid_free(orc_grid *g) { free(g->start); free(g->items); }

/* Same outputs as orc_forces_brute. Returns 0, or -1 if a periodic dimension
 * has fewer than 3 cells. */
int orc_forces_cells(const orc_params *p, long nv, const double *pos, long nw, const double *wall,
                     double *f, double *pe, double *pe_w, double *vir, long long *counts)
{
    const int dim = p->dim;
    const double rc2 = p->r_cut * p->r_cut;
    const double uc_vv = p->shift_energy ? u_cut(p->eps, p->sigma, p->r_cut) : 0.0;
    const double uc_vw = p->shift_energy ? u_cut(p->eps_w, p->sigma_w, p->r_cut) : 0.0;
    orc_grid gv, gw;
    if (grid_build(p, &gv, nv, pos) != 0) return -1;
    if (grid_build(p, &gw, nw, wall) != 0) { grid_free(&gv); return -1; }
    long long c_vv = 0, c_vw = 0;
    const int kz_lo = dim == 3 ? -1 : 0, kz_hi = dim == 3 ? 1 : 0;
#pragma omp parallel for schedule(static) reduction(+ : c_vv, c_vw)
    for (long i = 0; i < nv; ++i) {
        double fi[3] = {0.0, 0.0, 0.0}, u_vv = 0.0, u_vw = 0.0, w_vv = 0.0, w_vw = 0.0;
        long ci = cell_of(p, &gv, pos + i * dim);
        int c[3] = {(int)(ci % gv.n[0]), (int)((ci / gv.n[0]) % gv.n[1]), (int)(ci / ((long)gv.n[0] * gv.n[1]))};
        for (int kz = kz_lo; kz <= kz_hi; ++kz)
        for (int ky = -1; ky <= 1; ++ky)
        for (int kx = -1; kx <= 1; ++kx) {
            int k[3] = {kx, ky, kz}, q[3] = {0, 0, 0}, ok = 1;
            for (int a = 0; a < dim; ++a) {
                int m = c[a] + k[a];
                if (p->bc[a] == 0) m = (m + gv.n[a]) % gv.n[a];
                else if (m < 0 || m >= gv.n[a]) ok = 0;
                q[a] = m;
            }
            if (!ok) continue;
            long cj = ((long)q[2] * gv.n[1] + q[1]) * gv.n[0] + q[0];
            for (long s = gv.start[cj]; s < gv.start[cj + 1]; ++s) {
                long j = gv.items[s];
                if (j == i) continue;
                double d[3] = {0.0, 0.0, 0.0}, g, u, r2;
                for (int a = 0; a < dim; ++a) d[a] = pos[i * dim + a] - pos[j * dim + a];
                min_image(p, d);
                if (lj_pair(p->eps, p->sigma, rc2, uc_vv, dim, d, &g, &u, &r2)) {
                    for (int a = 0; a < dim; ++a) fi[a] += g * d[a];
                    u_vv += u; w_vv += g * r2; ++c_vv;
                }
            }
            for (long s = gw.start[cj]; s < gw.start[cj + 1]; ++s) {
                long w = gw.items[s];
                double d[3] = {0.0, 0.0, 0.0}, g, u, r2;
                for (int a = 0; a < dim; ++a) d[a] = pos[i * dim + a] - wall[w * dim + a];
                min_image(p, d);
                if (lj_pair(p->eps_w, p->sigma_w, rc2, uc_vw, dim, d, &g, &u, &r2)) {
                    for (int a = 0; a < dim; ++a) fi[a] += g * d[a];
                    u_vw += u; w_vw += g * r2; ++c_vw;
                }
            }
        }
        for (int a = 0; a < dim; ++a) f[i * dim + a] = fi[a];
        if (pe) pe[i] = 0.5 * u_vv + u_vw;
        if (pe_w) pe_w[i] = u_vw;
        if (vir) vir[i] = 0.5 * w_vv + w_vw;
    }
    if (counts) { counts[0] = c_vv; counts[1] = c_vw; }
    grid_free(&gv); grid_free(&gw);
    return 0;
}

/* ---- a5 energies ------------------------------------------------------ */
/* K = sum_i 1/2 m |v_i|^2 (plain left-to-right sum). */
double orc_kinetic(const orc_params *p, long nv, const double *vel)
{
    double k = 0.0;
    for (long i = 0; i < nv; ++i) {
        double v2 = 0.0;
        for (int a = 0; a < p->dim; ++a) v2 += vel[i * p->dim + a] * vel[i * p->dim + a];
        k += 0.5 * p->mass * v2;
    }
    return k;
}

static int forces(const orc_params *p, int use_cells, long nv, const double *pos, long nw, const double *wall,
                  double *f, double *pe, double *pe_w, double *vir, long long *counts)
{
    if (use_cells) return orc_forces_cells(p, nv, pos, nw, wall, f, pe, pe_w, vir, counts);
    orc_forces_brute(p, nv, pos, nw, wall, f, pe, pe_w, vir, counts);
    return 0;
}

/* ---- c.3 time stepping (kick-drift-kick form of PAPER.md:79-80, :88) --- */
/* Advances pos/vel in place by n_steps; f, pe, pe_w, vir (each may not be NULL
 * except vir) hold f(t), pe(t) at the final step on return.  f(0) is evaluated
 * here first (the caller's f is ignored on entry).  If hist != NULL it
 * receives (n_steps + 1) rows of {K, U_vv, U_vw, pairs_vv_ordered, pairs_vw}
 * for steps 0..n_steps.  Returns 0; -1 cell grid invalid; -2 a particle left
 * the box after one bounce (reading A4: one bounce per step at most). */
int orc_run(const orc_params *p, int use_cells, long nv, double *pos, double *vel, long nw, const double *wall,
            long n_steps, double *f, double *pe, double *pe_w, double *vir, double *hist)
{
    const int dim = p->dim;
    const double hk = p->dt / (2.0 * p->mass);
    long long counts[2];
    if (forces(p, use_cells, nv, pos, nw, wall, f, pe, pe_w, vir, counts) != 0) return -1;
    for (long step = 0;; ++step) {
        if (hist) {
            double uw = 0.0, ut = 0.0;
            for (long i = 0; i < nv; ++i) { uw += pe_w[i]; ut += pe[i]; }
            hist[step * 5 + 0] = orc_kinetic(p, nv, vel);
            hist[step * 5 + 1] = ut - uw;
            hist[step * 5 + 2] = uw;
            hist[step * 5 + 3] = (double)counts[0];
            hist[step * 5 + 4] = (double)counts[1];
        }
        if (step == n_steps) break;
        int bad = 0;
        for (long i = 0; i < nv; ++i) {
            double ro[3] = {0, 0, 0}, rn[3] = {0, 0, 0}, vh[3] = {0, 0, 0};
            for (int a = 0; a < dim; ++a) {
                ro[a] = pos[i * dim + a];
                vh[a] = vel[i * dim + a] + hk * f[i * dim + a];             /* F2: v(t + dt/2) */
                rn[a] = ro[a] + p->dt * vh[a];                              /* F2: r(t + dt)   */
            }
            if (p->prism) {
                /* geometric pore walls: one specular bounce per closed face whose rectangle the straight path
                 * r(t) -> r(t + dt) crosses; faces are visited in the order -x, +x, -y, +y, (-z, +z) */
                for (int a = 0; a < dim; ++a)
                    for (int sgn = -1; sgn <= 1; sgn += 2) {
                        if (a == p->prism_axis && sgn == 1) continue;             /* the open face */
                        const double w = p->prism_c[a] + sgn * p->prism_h[a];
                        if ((ro[a] - w) * (rn[a] - w) < 0.0) {
                            const double t = (w - ro[a]) / (rn[a] - ro[a]);
                            int inside = 1;
                            for (int b = 0; b < dim; ++b)
                                if (b != a && fabs(ro[b] + t * (rn[b] - ro[b]) - p->prism_c[b]) > p->prism_h[b]) inside = 0;
                            if (inside) { rn[a] = 2.0 * w - rn[a]; vh[a] = -vh[a]; }
                        }
                    }
            }
            for (int a = 0; a < dim; ++a) {
                double v = vh[a], r = rn[a];
                const double L = p->L[a];
                if (p->bc[a] == 0) {                                    /* periodic wrap into [0, L) */
                    r = r - L * floor(r / L);
                    if (r >= L) r = r - L;
                } else {                                                /* specular reflection */
                    if (r < 0.0) { r = -r; v = -v; }
                    else if (r > L) { r = 2.0 * L - r; v = -v; }
                    if (r < 0.0 || r > L) bad = 1;
                }
                vel[i * dim + a] = v;
                pos[i * dim + a] = r;
            }
        }
        if (bad) return -2;
        if (forces(p, use_cells, nv, pos, nw, wall, f, pe, pe_w, vir, counts) != 0) return -1;   /* F1 */
        for (long i = 0; i < nv; ++i)
            for (int a = 0; a < dim; ++a)
                vel[i * dim + a] = vel[i * dim + a] + hk * f[i * dim + a];                       /* F3 */
        if (p->tau_b > 0.0) {                                                                    /* F4 */
            /* Berendsen: v <- lambda v, lambda = sqrt(1 + (dt / tau_B)(T_0 / T - 1)), T = 2K / (d N) with k_B = 1
             * (the paper names lambda(t) and tau_B but prints no formula: reading A9 / NEXT-1 of DESIGN.md) */
            const double T = 2.0 * orc_kinetic(p, nv, vel) / ((double)dim * (double)nv);
            if (T > 0.0) {
                const double lambda = sqrt(1.0 + (p->dt / p->tau_b) * (p->t_target / T - 1.0));
                for (long i = 0; i < nv * dim; ++i) vel[i] = lambda * vel[i];
            }
        }
    }
    return 0;
}

int orc_sizeof_params(void) { return (int)sizeof(orc_params); }
