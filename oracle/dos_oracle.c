/* dos_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of what the hot path computes, written from the paper
 * (/root/reference/PAPER.md, Norris & Liu, arXiv 1811.12391) and the readings listed in DESIGN.md
 * ("Readings of the paper", R1..R18 = SURVEY.md 8(c) S1..S18). Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load this library. It shares no source,
 * header, table or helper with the CUDA library under paper_1811_12391_b200/csrc/.
 *
 * Steps, in the paper's order:
 *   orc_harmonics        real Schmidt semi-normalised harmonics Y_lm (reading R10; PAPER.md:41
 *                        "expressed as a function of Legendre expansion")
 *   orc_uncollided       ray-traced uncollided fluence phi_u ("computable with a
 *                        ray-tracing algorithm"; "per source particle")
 *   orc_first_collision  first-collision source moments
 *   orc_sweep            one transport sweep of eq. 2's left side for a frozen right side
 *                        (PAPER.md:39-41), scalar/moment fluence by eq. 3,
 *                        diamond difference + set-to-zero fixup (north_star; reading R3)
 *   orc_solve            group cascade + source iteration (PAPER.md:39 one-sided g' sum; R1, R5)
 *   orc_dose             fluence-to-dose weighting
 *
 * Pins (tests/test_oracle_pins.py): analytic point-source fluence, infinite-medium closed form,
 * particle balance, quadrature/harmonic orthogonality, mirror symmetry, brute-force 4^3 linear
 * system, 1-cell and 1-D diamond-difference closed forms, independent DDA ray walk.
 * Parity unpinned: accuracy against Monte Carlo (Tables 1-5) -- MCNP6 and its data are
 * not in the container.
 *
 * Layout: every field is [..][nz][ny][nx], x fastest. Moments are [M][Nv], lm = l(l+1)+m.
 * Threads: OpenMP over the independent angles of one octant only; each angle's sweep and the
 * accumulation order over angles are fixed, so results do not depend on the thread count.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t nx, ny, nz;
    double dx, dy, dz;
    double x0, y0, z0;
} orc_mesh;

#define ORC_PI 3.14159265358979323846

/* ---------------------------------------------------------------- O0 harmonics (reading R10) -- */
/* Polar axis z. Y_l0 = P_l(xi); m>0: Y_l,+m = sqrt(2 (l-m)!/(l+m)!) P_l^m(xi) cos(m phi),
 * Y_l,-m = same * sin(m phi); phi = atan2(eta, mu); P_l^m WITHOUT Condon-Shortley phase. */
void orc_harmonics(double mu, double eta, double xi, int L, double *y)
{
    double phi = atan2(eta, mu);
    double s2 = 1.0 - xi * xi;
    if (s2 < 0.0) s2 = 0.0;
    double s = sqrt(s2);
    int pole = (s2 == 0.0);
    for (int m = 0; m <= L; ++m) {
        /* P_m^m = (2m-1)!! (1-xi^2)^{m/2} */
        double pmm = 1.0;
        for (int t = 1; t <= m; ++t) pmm *= (2.0 * t - 1.0) * s;
        double plm2 = 0.0, plm1 = 0.0;
        for (int l = m; l <= L; ++l) {
            double plm;
            if (l == m) plm = pmm;
            else if (l == m + 1) plm = (2.0 * m + 1.0) * xi * pmm;
            else plm = ((2.0 * l - 1.0) * xi * plm1 - (l + m - 1.0) * plm2) / (double)(l - m);
            plm2 = plm1; plm1 = plm;
            if (m == 0) {
                y[l * (l + 1)] = plm;
            } else {
                double ratio = 1.0;               /* (l-m)!/(l+m)! */
                for (int t = l - m + 1; t <= l + m; ++t) ratio /= (double)t;
                double nrm = sqrt(2.0 * ratio);
                double c = pole ? 1.0 : cos(m * phi);
                double sn = pole ? 0.0 : sin(m * phi);
                y[l * (l + 1) + m] = nrm * plm * c;
                y[l * (l + 1) - m] = nrm * plm * sn;
            }
        }
    }
}

/* ------------------------------------------------------- O1 uncollided fluence (R6-R9) -------- */
static int cmp_double(const void *a, const void *b)
{
    double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

/* Radiological path lengths per material from the point `s` to the point `c` through the mesh:
 * parametric ray-grid method: collect alpha of every grid plane crossing, sort, identify the cell of
 * each interval by its midpoint. len_mat[n_mat] receives the summed geometric length per material;
 * returns total in-mesh length. The part of the segment outside the mesh contributes nothing (R9). */
static double path_lengths(const orc_mesh *ms, const uint8_t *mat, int n_mat, const double s[3],
                           const double c[3], double *len_mat, double *alpha_buf)
{
    double d[3] = {c[0] - s[0], c[1] - s[1], c[2] - s[2]};
    double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    int n[3] = {ms->nx, ms->ny, ms->nz};
    double h[3] = {ms->dx, ms->dy, ms->dz};
    double o[3] = {ms->x0, ms->y0, ms->z0};
    for (int m = 0; m < n_mat; ++m) len_mat[m] = 0.0;
    double amin = 0.0, amax = 1.0;
    for (int ax = 0; ax < 3; ++ax) {
        double lo = o[ax], hi = o[ax] + n[ax] * h[ax];
        if (d[ax] == 0.0) {
            if (s[ax] < lo || s[ax] > hi) return 0.0;
        } else {
            double a0 = (lo - s[ax]) / d[ax], a1 = (hi - s[ax]) / d[ax];
            double en = a0 < a1 ? a0 : a1, ex = a0 < a1 ? a1 : a0;
            if (en > amin) amin = en;
            if (ex < amax) amax = ex;
        }
    }
    if (!(amin < amax)) return 0.0;
    int cnt = 0;
    alpha_buf[cnt++] = amin;
    alpha_buf[cnt++] = amax;
    for (int ax = 0; ax < 3; ++ax) {
        if (d[ax] == 0.0) continue;
        for (int p = 0; p <= n[ax]; ++p) {
            double a = (o[ax] + p * h[ax] - s[ax]) / d[ax];
            if (a > amin && a < amax) alpha_buf[cnt++] = a;
        }
    }
    qsort(alpha_buf, (size_t)cnt, sizeof(double), cmp_double);
    double total = 0.0;
    for (int t = 0; t + 1 < cnt; ++t) {
        double a = alpha_buf[t], b = alpha_buf[t + 1];
        if (!(b > a)) continue;
        double mid = 0.5 * (a + b);
        int idx[3];
        for (int ax = 0; ax < 3; ++ax) {
            double p = s[ax] + mid * d[ax];
            int q = (int)floor((p - o[ax]) / h[ax]);
            if (q < 0) q = 0;
            if (q > n[ax] - 1) q = n[ax] - 1;
            idx[ax] = q;
        }
        double len = (b - a) * r;
        int m = mat[((size_t)idx[2] * n[1] + idx[1]) * n[0] + idx[0]];
        len_mat[m] += len;
        total += len;
    }
    return total;
}

/* Inside test of the collimated beam (reading R8): rectangular pyramid about `axis`, hard edge,
 * tested at the voxel centre, boundary inclusive. */
static int inside_beam(const double d[3], const double axis[3], const double up[3], double tan_fan,
                       double tan_cone, int isotropic)
{
    if (isotropic) return 1;
    double a = d[0] * axis[0] + d[1] * axis[1] + d[2] * axis[2];
    if (!(a > 0.0)) return 0;
    double u = d[0] * up[0] + d[1] * up[1] + d[2] * up[2];
    double side[3] = {axis[1] * up[2] - axis[2] * up[1], axis[2] * up[0] - axis[0] * up[2],
                      axis[0] * up[1] - axis[1] * up[0]};
    double v = d[0] * side[0] + d[1] * side[1] + d[2] * side[2];
    return fabs(u) <= a * tan_cone && fabs(v) <= a * tan_fan;
}

/* phi_u^g(c) = S_g exp(-tau_g) / (4 pi r^2) inside the beam, 0 outside (R7), for ONE voxel.
 * out[g] (stride `stride` doubles between groups). Returns 1 if the source sits on the voxel centre. */
static int uncollided_cell(const orc_mesh *ms, const uint8_t *mat, int n_mat, int G, const double *sigma_t,
                           const double *pos, const double *axis, const double *up, double tan_fan,
                           double tan_cone, int isotropic, const double *spectrum, long long cell,
                           double *out, size_t stride, double *path_total, double *len_mat, double *abuf)
{
    int i = (int)(cell % ms->nx), j = (int)((cell / ms->nx) % ms->ny),
        k = (int)(cell / ((long long)ms->nx * ms->ny));
    double c[3] = {ms->x0 + (i + 0.5) * ms->dx, ms->y0 + (j + 0.5) * ms->dy, ms->z0 + (k + 0.5) * ms->dz};
    double d[3] = {c[0] - pos[0], c[1] - pos[1], c[2] - pos[2]};
    double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    if (r2 < 1e-18) return 1;
    if (!inside_beam(d, axis, up, tan_fan, tan_cone, isotropic)) {
        for (int g = 0; g < G; ++g) out[(size_t)g * stride] = 0.0;
        if (path_total) *path_total = 0.0;
        return 0;
    }
    double tot = path_lengths(ms, mat, n_mat, pos, c, len_mat, abuf);
    if (path_total) *path_total = tot;
    for (int g = 0; g < G; ++g) {
        double tau = 0.0;
        for (int m = 0; m < n_mat; ++m) tau += sigma_t[(size_t)m * G + g] * len_mat[m];
        out[(size_t)g * stride] = spectrum[g] * exp(-tau) / (4.0 * ORC_PI * r2);
    }
    return 0;
}

/* All voxels. sigma_t [n_mat][G]; phi_u out [G][Nv]; optional path_total out [Nv] (in-mesh length). */
int orc_uncollided(const orc_mesh *ms, const uint8_t *mat, int n_mat, int G, const double *sigma_t,
                   const double *pos, const double *axis, const double *up, double tan_fan,
                   double tan_cone, int isotropic, const double *spectrum, double *phi_u,
                   double *path_total)
{
    size_t nv = (size_t)ms->nx * ms->ny * ms->nz;
    int err = 0;
#pragma omp parallel
    {
        double *len_mat = (double *)malloc(sizeof(double) * (size_t)n_mat);
        double *abuf = (double *)malloc(sizeof(double) * (size_t)(ms->nx + ms->ny + ms->nz + 8));
#pragma omp for schedule(dynamic, 64)
        for (long long cell = 0; cell < (long long)nv; ++cell)
            if (uncollided_cell(ms, mat, n_mat, G, sigma_t, pos, axis, up, tan_fan, tan_cone, isotropic,
                                spectrum, cell, phi_u + cell, nv, path_total ? path_total + cell : NULL,
                                len_mat, abuf))
                err = 1;
        free(len_mat);
        free(abuf);
    }
    return err;
}

/* The same for a list of voxels (flat indices cells[n_cells]); phi_u out [G][n_cells]. Used to check
 * sampled voxels of meshes too large to trace in full. */
int orc_uncollided_cells(const orc_mesh *ms, const uint8_t *mat, int n_mat, int G, const double *sigma_t,
                         const double *pos, const double *axis, const double *up, double tan_fan,
                         double tan_cone, int isotropic, const double *spectrum, const long long *cells,
                         long long n_cells, double *phi_u)
{
    int err = 0;
#pragma omp parallel
    {
        double *len_mat = (double *)malloc(sizeof(double) * (size_t)n_mat);
        double *abuf = (double *)malloc(sizeof(double) * (size_t)(ms->nx + ms->ny + ms->nz + 8));
#pragma omp for schedule(dynamic, 16)
        for (long long t = 0; t < n_cells; ++t)
            if (uncollided_cell(ms, mat, n_mat, G, sigma_t, pos, axis, up, tan_fan, tan_cone, isotropic,
                                spectrum, cells[t], phi_u + t, (size_t)n_cells, NULL, len_mat, abuf))
                err = 1;
        free(len_mat);
        free(abuf);
    }
    return err;
}

/* ------------------------------------------------------------ O2 first-collision moments ------ */
/* Q_fc^g[lm](c) = Y_lm(Omega_r(c)) * sum_{g'<=g} sigma_sl[m(c)][l][g'->g] phi_u^{g'}(c)
 * sigma_s [n_mat][n_leg+1][G from][G to]; q out [M][Nv] for the ONE group g; ADDS into q. */
void orc_first_collision(const orc_mesh *ms, const uint8_t *mat, int G, int n_leg, int L,
                         const double *sigma_s, const double *pos, const double *phi_u, int g,
                         double *q)
{
    size_t nv = (size_t)ms->nx * ms->ny * ms->nz;
    int M = (L + 1) * (L + 1);
#pragma omp parallel for schedule(static)
    for (long long cell = 0; cell < (long long)nv; ++cell) {
        int i = (int)(cell % ms->nx), j = (int)((cell / ms->nx) % ms->ny),
            k = (int)(cell / ((long long)ms->nx * ms->ny));
        double d[3] = {ms->x0 + (i + 0.5) * ms->dx - pos[0], ms->y0 + (j + 0.5) * ms->dy - pos[1],
                       ms->z0 + (k + 0.5) * ms->dz - pos[2]};
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        double y[64];
        orc_harmonics(d[0] / r, d[1] / r, d[2] / r, L, y);
        int m = mat[cell];
        for (int l = 0; l <= L; ++l) {
            double s = 0.0;
            for (int gp = 0; gp <= g; ++gp)
                s += sigma_s[(((size_t)m * (n_leg + 1) + l) * G + gp) * G + g] *
                     phi_u[(size_t)gp * nv + cell];
            for (int mm = -l; mm <= l; ++mm) q[(size_t)(l * (l + 1) + mm) * nv + cell] += y[l * (l + 1) + mm] * s;
        }
    }
    (void)M;
}

/* --------------------------------------------------------------------- O4 one sweep ----------- */
/* Cell update: diamond difference with set-to-zero fixup WITH rebalance (reading R3, R12).
 * psi_in[3], c[3] = 2|Omega_d|/Delta_d, returns psi_c, writes psi_out[3]. (Not static: dos_oracle_blocked.c, the
 * second loop arrangement used for full-size golden runs, calls this same function.) */
double orc_dd_cell(double q, double sig_t, const double c[3], const double pin[3], double pout[3])
{
    int fixed[3] = {0, 0, 0};
    double pc = 0.0;
    for (;;) {
        double num = q, den = sig_t;
        for (int d = 0; d < 3; ++d) {
            if (fixed[d]) num += 0.5 * c[d] * pin[d];
            else { num += c[d] * pin[d]; den += c[d]; }
        }
        pc = num / den;
        int added = 0, neg[3] = {0, 0, 0};
        for (int d = 0; d < 3; ++d) {
            if (fixed[d]) { pout[d] = 0.0; continue; }
            pout[d] = 2.0 * pc - pin[d];
            if (pout[d] < 0.0) neg[d] = 1;
        }
        for (int d = 0; d < 3; ++d)
            if (neg[d]) { fixed[d] = 1; added = 1; }
        if (!added) break;
    }
    for (int d = 0; d < 3; ++d) if (fixed[d]) pout[d] = 0.0;
    return pc;
}

/* Sweep one ordinate n over the whole mesh in upwind order (plain nested loops).
 * Q [M][Nv] frozen source moments; coef[M] = (2l+1) Y_lm(Omega_n); psi_c out [Nv].
 * bnd_in (may be NULL = vacuum): incoming boundary fluxes for this angle, three arrays packed as
 * [ny*nz | nx*nz | nx*ny]; bnd_out (may be NULL): outgoing boundary fluxes, same packing. */
static void sweep_angle(const orc_mesh *ms, const uint8_t *mat, const double *sig_t_g, double mu,
                        double eta, double xi, int M, const double *coef, const double *Q,
                        double *psi_c, const double *bnd_in, double *bnd_out, double *fy, double *fz)
{
    int nx = ms->nx, ny = ms->ny, nz = ms->nz;
    size_t nv = (size_t)nx * ny * nz;
    double c[3] = {2.0 * fabs(mu) / ms->dx, 2.0 * fabs(eta) / ms->dy, 2.0 * fabs(xi) / ms->dz};
    int di = mu > 0 ? 1 : -1, dj = eta > 0 ? 1 : -1, dk = xi > 0 ? 1 : -1;
    const double *bx = bnd_in, *by = bnd_in ? bnd_in + (size_t)ny * nz : NULL,
                 *bz = bnd_in ? bnd_in + (size_t)ny * nz + (size_t)nx * nz : NULL;
    double *ox = bnd_out, *oy = bnd_out ? bnd_out + (size_t)ny * nz : NULL,
           *oz = bnd_out ? bnd_out + (size_t)ny * nz + (size_t)nx * nz : NULL;
    /* fz[ny][nx]: z-face flux entering the current k-plane; fy[nx]: y-face flux entering row j */
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) fz[(size_t)j * nx + i] = bz ? bz[(size_t)j * nx + i] : 0.0;
    for (int kk = 0; kk < nz; ++kk) {
        int k = dk > 0 ? kk : nz - 1 - kk;
        for (int i = 0; i < nx; ++i) fy[i] = by ? by[(size_t)k * nx + i] : 0.0;
        for (int jj = 0; jj < ny; ++jj) {
            int j = dj > 0 ? jj : ny - 1 - jj;
            double fx = bx ? bx[(size_t)k * ny + j] : 0.0;
            for (int ii = 0; ii < nx; ++ii) {
                int i = di > 0 ? ii : nx - 1 - ii;
                size_t cell = ((size_t)k * ny + j) * nx + i;
                double q = 0.0;
                for (int lm = 0; lm < M; ++lm) q += coef[lm] * Q[(size_t)lm * nv + cell];
                double pin[3] = {fx, fy[i], fz[(size_t)j * nx + i]}, pout[3];
                psi_c[cell] = orc_dd_cell(q, sig_t_g[mat[cell]], c, pin, pout);
                fx = pout[0];
                fy[i] = pout[1];
                fz[(size_t)j * nx + i] = pout[2];
            }
            if (ox) ox[(size_t)k * ny + j] = fx;
        }
        if (oy) for (int i = 0; i < nx; ++i) oy[(size_t)k * nx + i] = fy[i];
    }
    if (oz) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) oz[(size_t)j * nx + i] = fz[(size_t)j * nx + i];
}

static size_t bnd_size(const orc_mesh *ms)
{
    return (size_t)ms->ny * ms->nz + (size_t)ms->nx * ms->nz + (size_t)ms->nx * ms->ny;
}

/* phi_new[lm](c) = sum_n w_n Y_lm(Omega_n) psi_c,n(c)   (eq. 3 is the lm = 0 row)
 * Q [M][Nv]; phi_new out [M][Nv]; sig_t_g [n_mat] for this group.
 * reflective != 0: incoming boundary flux of angle n = outgoing flux of its mirror image stored in
 *   bnd_state [n_ang][bnd] by the previous call (lagged); bnd_state is updated. (oracle-only, pin 2)
 * leakage (may be NULL): sum over boundary faces of w_n |Omega_n . n| psi_out A  (oracle-only, pin 3)
 * psi_all (may be NULL): [n_ang][Nv] angular flux at cell centres (for the brute-force pin).
 * phi_abs (may be NULL): [Nv] sum_n w_n |psi_c,n(c)|, the size of the terms of eq. 3 -- a diagnostic
 *   for the parity tests (conditioning of phi[00] where angular fluxes of both signs cancel); it does
 *   not enter any result. */
int orc_sweep(const orc_mesh *ms, const uint8_t *mat, const double *sig_t_g, int n_ang,
              const double *mu, const double *eta, const double *xi, const double *w, int L,
              const double *Q, double *phi_new, int reflective, double *bnd_state, double *leakage,
              double *psi_all, double *phi_abs)
{
    int nx = ms->nx, ny = ms->ny, nz = ms->nz;
    size_t nv = (size_t)nx * ny * nz, nb = bnd_size(ms);
    int M = (L + 1) * (L + 1);
    double *ylm = (double *)malloc(sizeof(double) * (size_t)n_ang * M);
    for (int n = 0; n < n_ang; ++n) orc_harmonics(mu[n], eta[n], xi[n], L, ylm + (size_t)n * M);
    double *bnd_new = NULL;
    if (reflective || leakage) bnd_new = (double *)calloc((size_t)n_ang * nb, sizeof(double));
    memset(phi_new, 0, sizeof(double) * (size_t)M * nv);
    double *psi = psi_all ? psi_all : (double *)malloc(sizeof(double) * (size_t)n_ang * nv);
    if (!ylm || !psi || ((reflective || leakage) && !bnd_new)) return -1;

#pragma omp parallel
    {
        double *coef = (double *)malloc(sizeof(double) * (size_t)M);
        double *fy = (double *)malloc(sizeof(double) * (size_t)nx);
        double *fz = (double *)malloc(sizeof(double) * (size_t)nx * ny);
        double *bin = reflective ? (double *)malloc(sizeof(double) * nb) : NULL;
#pragma omp for schedule(dynamic, 1)
        for (int n = 0; n < n_ang; ++n) {
            for (int l = 0; l <= L; ++l)
                for (int m = -l; m <= l; ++m)
                    coef[l * (l + 1) + m] = (2.0 * l + 1.0) * ylm[(size_t)n * M + l * (l + 1) + m];
            if (reflective) {
                /* mirror images of Omega_n across the x, y and z faces */
                int mx = -1, my = -1, mz = -1;
                for (int p = 0; p < n_ang; ++p) {
                    if (mu[p] == -mu[n] && eta[p] == eta[n] && xi[p] == xi[n]) mx = p;
                    if (mu[p] == mu[n] && eta[p] == -eta[n] && xi[p] == xi[n]) my = p;
                    if (mu[p] == mu[n] && eta[p] == eta[n] && xi[p] == -xi[n]) mz = p;
                }
                const double *sx = bnd_state + (size_t)mx * nb;
                const double *sy = bnd_state + (size_t)my * nb + (size_t)ny * nz;
                const double *sz = bnd_state + (size_t)mz * nb + (size_t)ny * nz + (size_t)nx * nz;
                memcpy(bin, sx, sizeof(double) * (size_t)ny * nz);
                memcpy(bin + (size_t)ny * nz, sy, sizeof(double) * (size_t)nx * nz);
                memcpy(bin + (size_t)ny * nz + (size_t)nx * nz, sz, sizeof(double) * (size_t)nx * ny);
            }
            sweep_angle(ms, mat, sig_t_g, mu[n], eta[n], xi[n], M, coef, Q, psi + (size_t)n * nv, bin,
                        bnd_new ? bnd_new + (size_t)n * nb : NULL, fy, fz);
        }
        free(coef); free(fy); free(fz); free(bin);
        /* discrete-to-moment, angles accumulated in index order for every cell */
#pragma omp for schedule(static)
        for (long long cell = 0; cell < (long long)nv; ++cell)
            for (int n = 0; n < n_ang; ++n) {
                double p = w[n] * psi[(size_t)n * nv + cell];
                for (int lm = 0; lm < M; ++lm) phi_new[(size_t)lm * nv + cell] += ylm[(size_t)n * M + lm] * p;
            }
        if (phi_abs) {
#pragma omp for schedule(static)
            for (long long cell = 0; cell < (long long)nv; ++cell) {
                double a = 0.0;
                for (int n = 0; n < n_ang; ++n) a += w[n] * fabs(psi[(size_t)n * nv + cell]);
                phi_abs[cell] = a;
            }
        }
    }
    if (leakage) {
        double lk = 0.0;
        for (int n = 0; n < n_ang; ++n) {
            const double *b = bnd_new + (size_t)n * nb;
            double sx = 0, sy = 0, sz = 0;
            for (size_t t = 0; t < (size_t)ny * nz; ++t) sx += b[t];
            for (size_t t = 0; t < (size_t)nx * nz; ++t) sy += b[(size_t)ny * nz + t];
            for (size_t t = 0; t < (size_t)nx * ny; ++t) sz += b[(size_t)ny * nz + (size_t)nx * nz + t];
            lk += w[n] * (fabs(mu[n]) * ms->dy * ms->dz * sx + fabs(eta[n]) * ms->dx * ms->dz * sy +
                          fabs(xi[n]) * ms->dx * ms->dy * sz);
        }
        *leakage = lk;
    }
    if (reflective) memcpy(bnd_state, bnd_new, sizeof(double) * (size_t)n_ang * nb);
    free(bnd_new);
    free(ylm);
    if (!psi_all) free(psi);
    return 0;
}

/* ------------------------------------------------------- O3 group cascade + source iteration --- */
/* for g = 0..G-1 (g = 0 highest energy; PAPER.md:39 one-sided g' sum, reading R1):
 *   Q_fix = q_ext^g (optional, [G][M][Nv]) + Q_fc^g (if phi_u != NULL) + sum_{g'<g} sigma_sl^{g'->g} phi_c^{g'}[lm]
 *   phi^(0) = 0; it = 1..n_iter: Q = Q_fix + sigma_sl^{g->g} phi^(it-1); phi^(it) = Sweep(Q)   (R5)
 * phi_c out [G][M][Nv]. leak out [G] (may be NULL): leakage of the LAST sweep of each group.
 * absorbed-source bookkeeping for the balance pin: src_last [G] (may be NULL) = sum_c V Q[00](c) of
 * the last sweep's source. phi_abs [G][Nv] (may be NULL): orc_sweep's diagnostic of the last sweep. */
/* n_iter_g (may be NULL): per-group iteration counts that replace n_iter (the counts a tolerance-stopped GPU run
 * reports, so that both sides do the same number of sweeps). conv out [G] (may be NULL): the
 * stopping measure of the last iteration of each group, max_c |phi00^(it) - phi00^(it-1)| / max_c |phi00^(it)|. */
int orc_solve_iters(const orc_mesh *ms, const uint8_t *mat, int n_mat, int G, int n_leg, int L,
                    const double *sigma_t, const double *sigma_s, int n_ang, const double *mu,
                    const double *eta, const double *xi, const double *w, const double *pos,
                    const double *phi_u, const double *q_ext, int n_iter, const int *n_iter_g, int reflective,
                    double *phi_c, double *leak, double *src_last, double *phi_abs, double *conv)
{
    size_t nv = (size_t)ms->nx * ms->ny * ms->nz, nb = bnd_size(ms);
    int M = (L + 1) * (L + 1);
    double *qfix = (double *)malloc(sizeof(double) * (size_t)M * nv);
    double *q = (double *)malloc(sizeof(double) * (size_t)M * nv);
    double *phi_old = (double *)malloc(sizeof(double) * (size_t)M * nv);
    double *sig_t_g = (double *)malloc(sizeof(double) * (size_t)n_mat);
    double *bnd = reflective ? (double *)malloc(sizeof(double) * (size_t)n_ang * nb) : NULL;
    if (!qfix || !q || !phi_old || !sig_t_g || (reflective && !bnd)) return -1;
    int rc = 0;
    for (int g = 0; g < G && rc == 0; ++g) {
        for (int m = 0; m < n_mat; ++m) sig_t_g[m] = sigma_t[(size_t)m * G + g];
        if (q_ext) memcpy(qfix, q_ext + (size_t)g * M * nv, sizeof(double) * (size_t)M * nv);
        else memset(qfix, 0, sizeof(double) * (size_t)M * nv);
        if (phi_u) orc_first_collision(ms, mat, G, n_leg, L, sigma_s, pos, phi_u, g, qfix);
        for (int gp = 0; gp < g; ++gp)
            for (int l = 0; l <= L; ++l)
                for (int mm = -l; mm <= l; ++mm) {
                    int lm = l * (l + 1) + mm;
                    const double *src = phi_c + ((size_t)gp * M + lm) * nv;
                    double *dst = qfix + (size_t)lm * nv;
                    for (size_t c = 0; c < nv; ++c)
                        dst[c] += sigma_s[(((size_t)mat[c] * (n_leg + 1) + l) * G + gp) * G + g] * src[c];
                }
        double *phi = phi_c + (size_t)g * M * nv;
        memset(phi_old, 0, sizeof(double) * (size_t)M * nv);
        if (bnd) memset(bnd, 0, sizeof(double) * (size_t)n_ang * nb);
        const int n_it = n_iter_g ? n_iter_g[g] : n_iter;
        for (int it = 1; it <= n_it && rc == 0; ++it) {
            for (int l = 0; l <= L; ++l)
                for (int mm = -l; mm <= l; ++mm) {
                    int lm = l * (l + 1) + mm;
                    for (size_t c = 0; c < nv; ++c)
                        q[(size_t)lm * nv + c] = qfix[(size_t)lm * nv + c] +
                            sigma_s[(((size_t)mat[c] * (n_leg + 1) + l) * G + g) * G + g] * phi_old[(size_t)lm * nv + c];
                }
            int last = (it == n_it);
            rc = orc_sweep(ms, mat, sig_t_g, n_ang, mu, eta, xi, w, L, q, phi, reflective, bnd,
                           (leak && last) ? &leak[g] : NULL, NULL,
                           (phi_abs && last) ? phi_abs + (size_t)g * nv : NULL);
            if (last && src_last) {
                double s = 0.0;
                for (size_t c = 0; c < nv; ++c) s += q[c];
                src_last[g] = s * ms->dx * ms->dy * ms->dz;
            }
            if (last && conv) {
                double dmax = 0.0, pmax = 0.0;
                for (size_t c = 0; c < nv; ++c) {
                    double d = fabs(phi[c] - phi_old[c]), a = fabs(phi[c]);
                    if (d > dmax) dmax = d;
                    if (a > pmax) pmax = a;
                }
                conv[g] = pmax > 0.0 ? dmax / pmax : 0.0;
            }
            memcpy(phi_old, phi, sizeof(double) * (size_t)M * nv);
        }
    }
    free(qfix); free(q); free(phi_old); free(sig_t_g); free(bnd);
    return rc;
}

/* The fixed-count form every config uses (reading R5): n_iter sweeps in every group, no convergence test. */
int orc_solve(const orc_mesh *ms, const uint8_t *mat, int n_mat, int G, int n_leg, int L,
              const double *sigma_t, const double *sigma_s, int n_ang, const double *mu,
              const double *eta, const double *xi, const double *w, const double *pos,
              const double *phi_u, const double *q_ext, int n_iter, int reflective, double *phi_c,
              double *leak, double *src_last, double *phi_abs)
{
    return orc_solve_iters(ms, mat, n_mat, G, n_leg, L, sigma_t, sigma_s, n_ang, mu, eta, xi, w, pos, phi_u, q_ext,
                           n_iter, NULL, reflective, phi_c, leak, src_last, phi_abs, NULL);
}

/* ------------------------------------------------------------------ O5 totals and dose -------- */
/* phi^g = phi_u^g + phi_c^g[00]; D(c) = sum_g K[m(c)][g] phi^g(c).
 * phi_c_moments [G][M][Nv]; phi_total out [G][Nv] (may be NULL); dose out [Nv]; accumulate adds. */
void orc_dose(const orc_mesh *ms, const uint8_t *mat, int G, int M, const double *kerma,
              const double *phi_u, const double *phi_c_moments, double *phi_total, double *dose,
              int accumulate)
{
    size_t nv = (size_t)ms->nx * ms->ny * ms->nz;
    for (size_t c = 0; c < nv; ++c) {
        double d = 0.0;
        for (int g = 0; g < G; ++g) {
            double p = (phi_u ? phi_u[(size_t)g * nv + c] : 0.0) + phi_c_moments[((size_t)g * M) * nv + c];
            if (phi_total) phi_total[(size_t)g * nv + c] = p;
            d += kerma[(size_t)mat[c] * G + g] * p;
        }
        dose[c] = accumulate ? dose[c] + d : d;
    }
}
