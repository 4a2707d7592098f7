/* dos_oracle_blocked.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A second loop arrangement of orc_solve (dos_oracle.c) for the full-size golden runs of configs 3-5
 * (tests/golden/make_golden.py): the SAME arithmetic in the SAME order per result, so its output is
 * bit-identical to the plain nested-loop oracle (tests/test_oracle_pins.py::test_blocked_variant_is_bit_identical
 * checks this on small meshes for every quadrature / P_L the configs use). Nothing here is a statement of the
 * method of its own: the cell update is orc_dd_cell and the first-collision source is orc_first_collision, both
 * from dos_oracle.c; what changes is only which loop is outside which, and how much memory is held:
 *
 *   plain                                         blocked
 *   ------------------------------------------    ------------------------------------------------------------
 *   q[M][Nv] built, then every angle streams it   a thread sweeps a chunk of <= ORC_CHUNK consecutive angles of one
 *   (one angle per thread)                        octant row by row; the row's source moments
 *                                                 Q = Q_fix + sigma_s^{g->g} phi_old are formed once per row and
 *                                                 shared by the chunk's angles (same products and sums, one
 *                                                 multiply and one add per value, as in orc_solve)
 *   q_n(c) = sum_lm coef[lm] Q[lm][c], lm         the same sum in the same lm order, written as a loop over the
 *   ascending from 0.0                            cells of a row inside the lm loop
 *   psi of ALL angles stored ([n_ang][Nv]), then  psi of one super-block of chunks stored; after each super-block
 *   phi[lm][c] += Y[n][lm] (w[n] psi[n][c]),      the same accumulation for its angles, n ascending; super-blocks
 *   n ascending                                   run in ascending angle order, so every phi[lm][c] sees the same
 *                                                 sequence of additions
 *
 * Vacuum boundaries only; no leakage tally, no reflective option (oracle-only pins use orc_solve).
 * Compiled with -ffp-contract=off like dos_oracle.c: no fused multiply-add changes a rounding.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <omp.h>

typedef struct {
    int32_t nx, ny, nz;
    double dx, dy, dz;
    double x0, y0, z0;
} orc_mesh;

#define ORC_CHUNK 4

void orc_harmonics(double mu, double eta, double xi, int L, double *y);
double orc_dd_cell(double q, double sig_t, const double c[3], const double pin[3], double pout[3]);
void orc_first_collision(const orc_mesh *ms, const uint8_t *mat, int G, int n_leg, int L, const double *sigma_s,
                         const double *pos, const double *phi_u, int g, double *q);

/* Sweep the angles n0..n0+cnt-1 (all with the same direction signs) over the whole mesh, row by row.
 * qfix, phi_old [M][Nv]; ss_gg [n_mat][L+1] = sigma_s^{g->g}; coef [cnt][M] = (2l+1) Y_lm; psi out [cnt][Nv].
 * Scratch: Qrow [M][nx], qrow [nx], fy [cnt][nx], fz [cnt][ny*nx]. */
static void sweep_chunk(const orc_mesh *ms, const uint8_t *mat, const double *sig_t_g, int cnt, const double *mu,
                        const double *eta, const double *xi, int L, const double *coef, const double *qfix,
                        const double *phi_old, const double *ss_gg, double *psi, double *Qrow, double *qrow,
                        double *fy, double *fz)
{
    const int nx = ms->nx, ny = ms->ny, nz = ms->nz, M = (L + 1) * (L + 1);
    const size_t nv = (size_t)nx * ny * nz;
    const int di = mu[0] > 0 ? 1 : -1, dj = eta[0] > 0 ? 1 : -1, dk = xi[0] > 0 ? 1 : -1;
    double c[ORC_CHUNK][3];
    for (int a = 0; a < cnt; ++a) {
        c[a][0] = 2.0 * fabs(mu[a]) / ms->dx; c[a][1] = 2.0 * fabs(eta[a]) / ms->dy; c[a][2] = 2.0 * fabs(xi[a]) / ms->dz;
    }
    for (size_t t = 0; t < (size_t)cnt * ny * nx; ++t) fz[t] = 0.0;                 /* vacuum */
    for (int kk = 0; kk < nz; ++kk) {
        const int k = dk > 0 ? kk : nz - 1 - kk;
        for (size_t t = 0; t < (size_t)cnt * nx; ++t) fy[t] = 0.0;
        for (int jj = 0; jj < ny; ++jj) {
            const int j = dj > 0 ? jj : ny - 1 - jj;
            const size_t row = ((size_t)k * ny + j) * nx;
            /* the row's source moments: Q = Q_fix + sigma_s^{g->g} phi_old (orc_solve's q array, this row only) */
            for (int l = 0; l <= L; ++l)
                for (int mm = -l; mm <= l; ++mm) {
                    const int lm = l * (l + 1) + mm;
                    const double *qf = qfix + (size_t)lm * nv + row, *po = phi_old + (size_t)lm * nv + row;
                    double *Qr = Qrow + (size_t)lm * nx;
                    for (int i = 0; i < nx; ++i) Qr[i] = qf[i] + ss_gg[(size_t)mat[row + i] * (L + 1) + l] * po[i];
                }
            for (int a = 0; a < cnt; ++a) {
                const double *cf = coef + (size_t)a * M;
                for (int i = 0; i < nx; ++i) qrow[i] = 0.0;
                for (int lm = 0; lm < M; ++lm) {
                    const double cl = cf[lm];
                    const double *Qr = Qrow + (size_t)lm * nx;
                    for (int i = 0; i < nx; ++i) qrow[i] += cl * Qr[i];
                }
                double *fya = fy + (size_t)a * nx, *fza = fz + ((size_t)a * ny + j) * nx, *ps = psi + (size_t)a * nv + row;
                double fx = 0.0;
                for (int ii = 0; ii < nx; ++ii) {
                    const int i = di > 0 ? ii : nx - 1 - ii;
                    double pin[3] = {fx, fya[i], fza[i]}, pout[3];
                    ps[i] = orc_dd_cell(qrow[i], sig_t_g[mat[row + i]], c[a], pin, pout);
                    fx = pout[0];
                    fya[i] = pout[1];
                    fza[i] = pout[2];
                }
            }
        }
    }
}

/* Same contract as orc_solve (dos_oracle.c) with reflective = 0 and no balance outputs. phi_c out [G][M][Nv];
 * phi_abs (may be NULL) [G][Nv] = sum_n w_n |psi_n| of each group's last sweep. */
int orc_solve_blocked(const orc_mesh *ms, const uint8_t *mat, int n_mat, int G, int n_leg, int L,
                      const double *sigma_t, const double *sigma_s, int n_ang, const double *mu, const double *eta,
                      const double *xi, const double *w, const double *pos, const double *phi_u, const double *q_ext,
                      int n_iter, double *phi_c, double *phi_abs)
{
    const int nx = ms->nx, ny = ms->ny, nz = ms->nz, M = (L + 1) * (L + 1);
    const size_t nv = (size_t)nx * ny * nz;
    /* chunks: maximal runs of <= ORC_CHUNK consecutive angles with identical direction signs */
    int *c0 = (int *)malloc(sizeof(int) * (size_t)(n_ang + 1));
    int n_chunk = 0;
    for (int n = 0; n < n_ang;) {
        int e = n + 1;
        while (e < n_ang && e - n < ORC_CHUNK && (mu[e] > 0) == (mu[n] > 0) && (eta[e] > 0) == (eta[n] > 0) &&
               (xi[e] > 0) == (xi[n] > 0)) ++e;
        c0[n_chunk++] = n;
        n = e;
    }
    c0[n_chunk] = n_ang;
    const int nth = omp_get_max_threads();
    double *ylm = (double *)malloc(sizeof(double) * (size_t)n_ang * M);
    double *coef = (double *)malloc(sizeof(double) * (size_t)n_ang * M);
    double *qfix = (double *)malloc(sizeof(double) * (size_t)M * nv);
    double *phi_old = (double *)malloc(sizeof(double) * (size_t)M * nv);
    double *sig_t_g = (double *)malloc(sizeof(double) * (size_t)n_mat);
    double *ss_gg = (double *)malloc(sizeof(double) * (size_t)n_mat * (L + 1));
    double *psi = (double *)malloc(sizeof(double) * (size_t)nth * ORC_CHUNK * nv);      /* one super-block */
    if (!c0 || !ylm || !coef || !qfix || !phi_old || !sig_t_g || !ss_gg || !psi) return -1;
    for (int n = 0; n < n_ang; ++n) {
        orc_harmonics(mu[n], eta[n], xi[n], L, ylm + (size_t)n * M);
        for (int l = 0; l <= L; ++l)
            for (int m = -l; m <= l; ++m)
                coef[(size_t)n * M + l * (l + 1) + m] = (2.0 * l + 1.0) * ylm[(size_t)n * M + l * (l + 1) + m];
    }
    int rc = 0;
    for (int g = 0; g < G && rc == 0; ++g) {
        for (int m = 0; m < n_mat; ++m) {
            sig_t_g[m] = sigma_t[(size_t)m * G + g];
            for (int l = 0; l <= L; ++l) ss_gg[(size_t)m * (L + 1) + l] = sigma_s[(((size_t)m * (n_leg + 1) + l) * G + g) * G + g];
        }
        if (q_ext) memcpy(qfix, q_ext + (size_t)g * M * nv, sizeof(double) * (size_t)M * nv);
        else memset(qfix, 0, sizeof(double) * (size_t)M * nv);
        if (phi_u) orc_first_collision(ms, mat, G, n_leg, L, sigma_s, pos, phi_u, g, qfix);
        /* downscatter: for every value the additions run over g' ascending, as in orc_solve */
#pragma omp parallel for schedule(static)
        for (int lm = 0; lm < M; ++lm) {
            int l = 0;
            while ((l + 1) * (l + 1) <= lm) ++l;
            double *dst = qfix + (size_t)lm * nv;
            for (int gp = 0; gp < g; ++gp) {
                const double *src = phi_c + ((size_t)gp * M + lm) * nv;
                for (size_t c = 0; c < nv; ++c)
                    dst[c] += sigma_s[(((size_t)mat[c] * (n_leg + 1) + l) * G + gp) * G + g] * src[c];
            }
        }
        double *phi = phi_c + (size_t)g * M * nv;
        memset(phi_old, 0, sizeof(double) * (size_t)M * nv);
        for (int it = 1; it <= n_iter && rc == 0; ++it) {
            const int last = (it == n_iter);
            double *pabs = (phi_abs && last) ? phi_abs + (size_t)g * nv : NULL;
            memset(phi, 0, sizeof(double) * (size_t)M * nv);
            if (pabs) memset(pabs, 0, sizeof(double) * nv);
            for (int sb = 0; sb < n_chunk; sb += nth) {
                const int sb_end = sb + nth < n_chunk ? sb + nth : n_chunk;
                int fail = 0;
#pragma omp parallel
                {
                    double *Qrow = (double *)malloc(sizeof(double) * (size_t)M * nx);
                    double *qrow = (double *)malloc(sizeof(double) * (size_t)nx);
                    double *fy = (double *)malloc(sizeof(double) * (size_t)ORC_CHUNK * nx);
                    double *fz = (double *)malloc(sizeof(double) * (size_t)ORC_CHUNK * nx * ny);
                    if (!Qrow || !qrow || !fy || !fz) {
#pragma omp atomic write
                        fail = 1;
                    }
#pragma omp barrier
                    if (!fail) {
#pragma omp for schedule(static, 1)
                        for (int ch = sb; ch < sb_end; ++ch) {
                            const int n0 = c0[ch], cnt = c0[ch + 1] - n0;
                            sweep_chunk(ms, mat, sig_t_g, cnt, mu + n0, eta + n0, xi + n0, L, coef + (size_t)n0 * M, qfix,
                                        phi_old, ss_gg, psi + (size_t)(ch - sb) * ORC_CHUNK * nv, Qrow, qrow, fy, fz);
                        }
                        /* discrete-to-moment of this super-block's angles, n ascending for every (lm, cell) */
#pragma omp for schedule(static)
                        for (long long blk = 0; blk < (long long)((nv + 255) / 256); ++blk) {
                            const size_t b0 = (size_t)blk * 256, b1 = b0 + 256 < nv ? b0 + 256 : nv;
                            double p[256];
                            for (int ch = sb; ch < sb_end; ++ch)
                                for (int n = c0[ch]; n < c0[ch + 1]; ++n) {
                                    const double *ps = psi + ((size_t)(ch - sb) * ORC_CHUNK + (n - c0[ch])) * nv;
                                    for (size_t c = b0; c < b1; ++c) p[c - b0] = w[n] * ps[c];
                                    for (int lm = 0; lm < M; ++lm) {
                                        const double y = ylm[(size_t)n * M + lm];
                                        double *dst = phi + (size_t)lm * nv;
                                        for (size_t c = b0; c < b1; ++c) dst[c] += y * p[c - b0];
                                    }
                                    if (pabs)
                                        for (size_t c = b0; c < b1; ++c) pabs[c] += w[n] * fabs(ps[c]);
                                }
                        }
                    }
                    free(Qrow); free(qrow); free(fy); free(fz);
                }
                if (fail) rc = -1;
            }
            memcpy(phi_old, phi, sizeof(double) * (size_t)M * nv);
        }
    }
    free(c0); free(ylm); free(coef); free(qfix); free(phi_old); free(sig_t_g); free(ss_gg); free(psi);
    return rc;
}
