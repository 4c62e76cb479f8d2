/* Tiny driver for tests/test_oracle_sanitizers.py: runs the oracle (oracle/md_oracle.c, compiled into this program with
 * -fsanitize=address,undefined) on a small periodic / reflecting case with walls, brute force and cell list, thermostat and
 * prism pore, so that an out-of-bounds access, a leak or undefined behaviour in it aborts the test.  Test infrastructure. */
#include "../oracle/md_oracle.c"
#include <stdio.h>

static double urand(unsigned long long *s)
{
    *s = *s * 6364136223846793005ull + 1442695040888963407ull;
    return (double)(*s >> 11) / 9007199254740992.0;
}

int main(void)
{
    orc_params p;
    memset(&p, 0, sizeof p);
    p.dim = 3;
    p.L[0] = 8.1; p.L[1] = 7.7; p.L[2] = 9.3;
    p.bc[0] = 0; p.bc[1] = 0; p.bc[2] = 1;
    p.eps = 0.7; p.sigma = 0.95; p.eps_w = 1.6; p.sigma_w = 0.9; p.r_cut = 2.5; p.shift_energy = 1;
    p.dt = 0.004; p.mass = 2.5; p.tau_b = 0.1; p.t_target = 0.8;
    p.prism = 1; p.prism_axis = 2; p.prism_c[0] = 4.0; p.prism_c[1] = 3.8; p.prism_c[2] = 4.6;
    p.prism_h[0] = 1.5; p.prism_h[1] = 1.5; p.prism_h[2] = 2.0;
    enum { NV = 150, NW = 17 };
    double *pos = malloc(sizeof(double) * NV * 3), *vel = malloc(sizeof(double) * NV * 3), *wall = malloc(sizeof(double) * NW * 3);
    double *f = malloc(sizeof(double) * NV * 3), *pe = malloc(sizeof(double) * NV), *pw = malloc(sizeof(double) * NV);
    double *vir = malloc(sizeof(double) * NV), *hist = malloc(sizeof(double) * 5 * 41);
    unsigned long long s = 12345;
    int n = 0;
    while (n < NV + NW) {                       /* random sequential placement, minimum separation 1 (plain distance) */
        double q[3] = {urand(&s) * p.L[0], urand(&s) * p.L[1], urand(&s) * p.L[2]};
        int ok = 1;
        for (int k = 0; k < n && ok; ++k) {
            const double *o = k < NV ? pos + 3 * k : wall + 3 * (k - NV);
            double d2 = 0;
            for (int a = 0; a < 3; ++a) d2 += (q[a] - o[a]) * (q[a] - o[a]);
            if (d2 < 1.0) ok = 0;
        }
        if (!ok) continue;
        double *dst = n < NV ? pos + 3 * n : wall + 3 * (n - NV);
        for (int a = 0; a < 3; ++a) dst[a] = q[a];
        ++n;
    }
    for (int k = 0; k < NV * 3; ++k) vel[k] = 1.2 * urand(&s) - 0.6;
    long long counts[2];
    orc_forces_brute(&p, NV, pos, NW, wall, f, pe, pw, vir, counts);
    long long cb = counts[0] + counts[1];
    if (orc_forces_cells(&p, NV, pos, NW, wall, f, pe, pw, vir, counts) != 0) return 2;
    if (cb != counts[0] + counts[1]) return 3;
    for (int cells = 0; cells < 2; ++cells)
        if (orc_run(&p, cells, NV, pos, vel, NW, wall, 40, f, pe, pw, vir, hist) != 0) return 4;
    printf("ok %lld pairs, K = %.6f\n", cb, orc_kinetic(&p, NV, vel));
    free(pos); free(vel); free(wall); free(f); free(pe); free(pw); free(vir); free(hist);
    return 0;
}
