// dos_api.cu -- the C ABI of include/dos.h: context, validation, workspace layout, host-side tables,
// and the launch sequence of the hot path. Kernels: dos_kernels.cu (ray trace, sources, dose),
// dos_sweep_umma.cu (transport sweep on the tensor-memory path) and dos_sweep_ffma.cu (its FFMA fallback).
// No code is shared with oracle/.
#include "../../include/dos.h"
#include "dos_internal.h"
#include "dos_kernels.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

struct Layout {
    size_t phi_u, phi_all, qfix, q, fy, fz, done, queue, items, items_u, mat, dose_acc, sig_t, sig_s, kerma, m2d, d2m, cdd,
        bm2d, bd2m, signs, errflag, bx, by, bz, phi00_old, conv, um, phi_u_sum, slot, total;
    int n_slots;
};

struct dos_ctx {
    dos_mesh mesh;
    int n_mat, G, n_leg, L, M, MP, n_ang, per_oct;
    int ntj, ntk, n_items, ag, n_grp, chunk, grid;     // FFMA sweep: (octant, tile) items, angles per warp, warps, flag chunk, CTAs
    int n_aux;                                         // aux warps of the FFMA sweep CTA
    int asplit, ag_pref, aux_pref;                     // angle split of an octant over CTAs; option overrides (0 = default)
    int contraction_pref;                              // 0 auto, 1 FFMA (dos_sweep_ffma.cu), 2 tensor memory (dos_sweep_umma.cu)
    bool umma, umma_ok;                                // the choice in force; the quadrature admits the tensor-memory sweep
    int n_items_u, grid_u;                             // tensor-memory sweep: (quad, tile) items, CTAs
    int ll_pref;                                       // FFMA sweep: flag-in-data face hand-off on small meshes (1 when the mesh admits it, 0 never)
    unsigned epoch;                                    // ... its launch counter (never 0)
    int two_per_sm;                                    // FFMA sweep: 64-register two-CTAs-per-SM variant (0 never, 1 from 4 items per SM, 2 always)
    size_t nv;
    cudaStream_t stream;
    const uint8_t *d_mat;        // current material grid (caller's or the workspace copy)
    char *ws;
    Layout lay;
    std::vector<float> h_cdd;    // [per_oct][4] diamond-difference coefficients (host copy: travels in the sweep's parameters)
    std::vector<int> band_lo;    // [G]: lowest g' with a non-zero sigma_s^{g'->g}
    int state;                   // 0 created, 1 uncollided done, 2 solved
    bool can_sum, summed;        // workspace holds the summed-source buffers; the current uncollided state is a sum
    std::vector<dos_source> srcs;   // sources of the position slots in use
    int n_slots, active;         // position slots of the workspace; slots the current uncollided state fills (1 unless dos_uncollided_batch)
    bool have_dose_acc;
    bool mat_checked;            // the current material grid has been through validate_material_kernel
    int refl;                    // reflective faces: bit 0 x, 1 y, 2 z (dos_set_boundary); 0 = vacuum
    bool profile, prof_open;
    std::vector<cudaEvent_t> ev;  // pairs (start, stop); kind in ev_kind
    std::vector<int> ev_kind;     // 0 sweep, 1 ray trace
    std::vector<cudaEvent_t> ev_pool;   // recycled events (creating one per launch would cost host time)
    double acc_ms[2];
    int64_t acc_n[2];
    int64_t launches;
    std::string err;
};

static thread_local std::string g_err;

static dos_status fail(dos_ctx *c, dos_status s, const std::string &msg)
{
    if (c) c->err = msg; else g_err = msg;
    return s;
}

#define CUDA_TRY(c, call)                                                                              \
    do {                                                                                               \
        cudaError_t e_ = (call);                                                                       \
        if (e_ != cudaSuccess)                                                                         \
            return fail((c), DOS_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_));        \
    } while (0)

// Real Schmidt semi-normalised harmonics, lm = l(l+1)+m, without trigonometry:
// sin^m(theta) cos(m phi) = Re (mu + i eta)^m, sin^m(theta) sin(m phi) = Im (mu + i eta)^m, and
// P_l^m(xi) = sin^m(theta) T_l^m(xi) with T_m^m = (2m-1)!!, T_{m+1}^m = (2m+1) xi T_m^m,
// (l-m) T_l^m = (2l-1) xi T_{l-1}^m - (l+m-1) T_{l-2}^m  (no Condon-Shortley phase; R10).
static void host_ylm(double mu, double eta, double xi, int L, double *y)
{
    double re = 1.0, im = 0.0, dfact = 1.0;
    for (int m = 0; m <= L; ++m) {
        if (m > 0) {
            double nre = re * mu - im * eta, nim = re * eta + im * mu;
            re = nre; im = nim;
            dfact *= (2.0 * m - 1.0);
        }
        double t2 = 0.0, t1 = 0.0;
        for (int l = m; l <= L; ++l) {
            double t;
            if (l == m) t = dfact;
            else if (l == m + 1) t = (2.0 * m + 1.0) * xi * t1;
            else t = ((2.0 * l - 1.0) * xi * t1 - (l + m - 1.0) * t2) / (double)(l - m);
            t2 = t1; t1 = t;
            if (m == 0) { y[l * (l + 1)] = t; continue; }
            double f = 2.0;                       // 2 (l-m)!/(l+m)!
            for (int s = l - m + 1; s <= l + m; ++s) f /= (double)s;
            double nrm = std::sqrt(f);
            y[l * (l + 1) + m] = nrm * t * re;
            y[l * (l + 1) - m] = nrm * t * im;
        }
    }
}

static size_t align_up(size_t v) { return (v + 255) & ~(size_t)255; }

// Meshes on which the FFMA sweep hands tile faces over as (value, epoch) pairs: few tiles (every tile waits on its
// upwind tile all the way, so the hand-off latency per hop is what the sweep costs) and at most 10 angles per octant
// (one polling lane per 16-byte piece of a step's inflow).
static bool ll_mesh(const dos_mesh *m, int per_oct)
{
    const int ntj = (m->ny + DOS_TJ - 1) / DOS_TJ, ntk = (m->nz + DOS_TK - 1) / DOS_TK;
    return 8 * ntj * ntk <= 1024 && 3 * per_oct <= 32;
}

// Workspace = n_slots "slots" (everything one source position owns: its uncollided fluence, all groups' moments, the
// sweep's source, face buffers, flags and boundary buffers; slot b starts slot bytes x b further on) followed by what the
// positions share (work queue and items, material copy, tables, summed-source buffers).
static Layout make_layout(const dos_mesh *m, int n_mat, int G, int n_leg, int L, int n_ang, int n_slots)
{
    Layout l;
    const bool summed = n_slots > 1;
    const size_t nv = (size_t)m->nx * m->ny * m->nz;
    const int MP = dos_mpad(L), per = n_ang / 8;
    const int ntj = (m->ny + DOS_TJ - 1) / DOS_TJ, ntk = (m->nz + DOS_TK - 1) / DOS_TK;
    const int KP = (MP + 7) & ~7, A8 = (per + 7) & ~7, NAP = (per + 15) & ~15, NMP = (MP + 15) & ~15;
    // tile-face buffers, one per (octant, tile), indexed by wavefront diagonal
    // (small meshes: room for (value, epoch) pairs -- the FFMA sweep's flag-in-data hand-off, dos_internal.h)
    const size_t pairs = ll_mesh(m, per) ? 2 : 1;
    const size_t fy = pairs * 8 * ntj * ntk * (m->nx + DOS_FACE_PAD) * per * DOS_TK;
    const size_t fz = pairs * 8 * ntj * ntk * (m->nx + DOS_FACE_PAD) * per * DOS_TJ;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
    // ---- per slot ----
    l.phi_u = take(sizeof(float) * G * nv);
    l.phi_all = take(sizeof(float) * G * nv * MP);
    l.qfix = take(sizeof(float) * nv * MP);
    l.q = take(sizeof(float) * nv * MP);
    l.fy = take(sizeof(float) * fy);
    l.fz = take(sizeof(float) * fz);
    l.done = take(sizeof(int) * (size_t)8 * ntj * ntk * 8);      // FFMA sweep: up to 8 angle parts per (octant, tile)
    // reflective boundaries (tensor-memory sweep): two halves (previous / current sweep) of the boundary outflow
    l.bx = take(sizeof(float) * (size_t)2 * 8 * per * m->nz * m->ny);
    l.by = take(sizeof(float) * (size_t)2 * 8 * ntk * (m->nx + DOS_FACE_PAD) * per * DOS_TK);
    l.bz = take(sizeof(float) * (size_t)2 * 8 * ntj * (m->nx + DOS_FACE_PAD) * per * DOS_TJ);
    l.phi00_old = take(sizeof(float) * nv);                       // tolerance-stopped solve: scalar fluence of the previous iterate
    l.slot = off;
    l.n_slots = n_slots;
    off = l.slot * (size_t)n_slots;
    // ---- shared ----
    l.queue = take(sizeof(int) * 4);
    l.items = take(sizeof(int) * (size_t)8 * ntj * ntk);
    l.items_u = take(sizeof(int) * (size_t)2 * ntj * ntk);
    l.mat = take(nv);
    l.dose_acc = take(sizeof(float) * nv);
    l.sig_t = take(sizeof(float) * G * n_mat);          // stored [G][n_mat]
    l.sig_s = take(sizeof(float) * (size_t)n_mat * (n_leg + 1) * G * G);
    l.kerma = take(sizeof(float) * n_mat * G);
    l.m2d = take(sizeof(float) * (size_t)n_ang * MP);
    l.d2m = take(sizeof(float) * (size_t)n_ang * MP);
    l.cdd = take(sizeof(float) * per * 4);
    l.bm2d = take(sizeof(float) * (size_t)2 * NAP * KP);
    l.bd2m = take(sizeof(float) * (size_t)2 * NMP * A8);
    l.signs = take(sizeof(unsigned) * (size_t)8 * MP);
    l.errflag = take(sizeof(int) * 4);
    l.conv = take(sizeof(int) * 4);
    // summed-source mode (dos_uncollided_sum): uncollided moments of all positions and their scalar sum
    l.um = summed ? take(sizeof(float) * G * nv * MP) : 0;
    l.phi_u_sum = summed ? take(sizeof(float) * G * nv) : 0;
    l.total = off;
    return l;
}

static dos_status check_inputs(const dos_mesh *mesh, const dos_xs *xs, const dos_quadrature *q, int P_L)
{
    if (!mesh || !xs || !q) return fail(nullptr, DOS_ERR_INVALID_ARG, "null argument");
    if (mesh->nx < 1 || mesh->ny < 1 || mesh->nz < 1 || !(mesh->dx > 0) || !(mesh->dy > 0) || !(mesh->dz > 0))
        return fail(nullptr, DOS_ERR_INVALID_ARG, "mesh sizes and spacings must be positive");
    if ((size_t)mesh->nx * mesh->ny * mesh->nz >= ((size_t)1 << 31))
        return fail(nullptr, DOS_ERR_UNSUPPORTED, "more than 2^31 voxels");
    if (xs->n_mat < 1 || xs->n_mat > DOS_MAX_MAT) return fail(nullptr, DOS_ERR_UNSUPPORTED, "n_mat must be 1..16");
    if (xs->n_group < 1 || xs->n_leg < 0 || !xs->sigma_t || !xs->sigma_s || !xs->kerma)
        return fail(nullptr, DOS_ERR_INVALID_ARG, "bad cross-section table");
    if (xs->n_group > DOS_MAX_G) return fail(nullptr, DOS_ERR_UNSUPPORTED, "more than 64 energy groups");
    if (P_L < 0 || P_L > xs->n_leg) return fail(nullptr, DOS_ERR_SHAPE, "P_L must be 0..n_leg");
    if (P_L > DOS_MAX_L) return fail(nullptr, DOS_ERR_UNSUPPORTED, "P_L > 5");
    if (q->n_ang < 8 || q->n_ang % 8 || !q->mu || !q->eta || !q->xi || !q->w)
        return fail(nullptr, DOS_ERR_INVALID_ARG, "n_ang must be a positive multiple of 8");
    if (dos_sweep_ffma_angles_per_warp(q->n_ang / 8, P_L, 0) == 0 && !dos_sweep_umma_supported(q->n_ang / 8, P_L))
        return fail(nullptr, DOS_ERR_UNSUPPORTED, "no sweep shape for this number of angles per octant");
    return DOS_OK;
}

// Choice and shape of the sweep for the current option values. Default: the tensor-memory sweep (dos_sweep_umma.cu) from
// P4 up (28 / 36 moments per cell: the two contractions are 70-80 % of the arithmetic) wherever the quadrature admits
// it, the FFMA sweep below (measured: S8/P3 on 256x256x64 2.9 ms per sweep against 3.7) and as the fallback.
static cudaError_t configure_sweep(dos_ctx *c)
{
    // flag-in-data hand-off: the pair buffers must not hold anything that reads as a current epoch (the workspace is the
    // caller's memory; the tensor-memory sweep, if it ran on this context, left plain floats there)
    if (ll_mesh(&c->mesh, c->per_oct))
        for (int b = 0; b < c->lay.n_slots; ++b) {
            cudaError_t e = cudaMemsetAsync(c->ws + (size_t)b * c->lay.slot + c->lay.fy, 0, c->lay.done - c->lay.fy, c->stream);
            if (e != cudaSuccess) return e;
        }
    const bool ffma_ok = dos_sweep_ffma_angles_per_warp(c->per_oct, c->L, 0) != 0;
    const bool want_umma = c->contraction_pref == 2 || (c->contraction_pref == 0 && c->umma_ok && c->MP >= 28 && c->per_oct >= 3) || !ffma_ok || c->refl != 0;
    if (want_umma) {
        if (!c->umma_ok) return cudaErrorInvalidValue;
        int grid = 0;
        cudaError_t e = dos_sweep_umma_grid(c->L, c->per_oct, c->n_mat, c->n_items_u, &grid);
        if (e != cudaSuccess) return e;
        c->grid_u = grid;
        c->umma = true;
        return cudaSuccess;
    }
    int as = c->asplit;
    if (as < 1 || c->per_oct % as) as = 1;
    const int ap = c->per_oct / as;
    int ag = dos_sweep_ffma_angles_per_warp(ap, c->L, c->ag_pref);
    if (ag == 0 || (c->ag_pref > 0 && ag != c->ag_pref)) return cudaErrorInvalidValue;
    int nx = dos_sweep_ffma_aux_warps(ap, c->L, ag, c->aux_pref);
    if (ap / ag + nx + 2 > 24) return cudaErrorInvalidValue;
    // Meshes with many work items per SM run the 64-register variant, several CTAs per SM (dos_sweep_ffma.cu: pick). A CTA
    // of at most 10 warps fits three times instead of twice: measured at config 4 (S8/P3, 256x256x64), 2 angles per warp
    // and 3 aux warps (5 + 3 + 2 warps, 3 CTAs per SM) 2.77 ms per sweep against 2.88 for 1 and 4 (16 warps, 2 CTAs);
    // 2 and 2: 2.79; 2 and 4 (11 warps, 2 CTAs): 3.24; 2 and 1: 3.37. Only when the caller has not fixed the shape.
    // (paper-shaped fine mesh, S6/P0: 1 angle per warp, 9 warps, 3 CTAs per SM 1.40 ms; 2 per warp, 6 warps, 5 CTAs 1.25; 3: 1.30)
    if (c->ag_pref == 0 && c->aux_pref == 0 && c->two_per_sm && c->MP <= 16 && ag == 1 && ap / ag + nx + 2 > 6) {
        int sms = 148, dev = 0;
        if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        const long items = (long)c->n_items * as;
        if (items >= 16L * sms)      // (128x128x64, 14 items per SM: 0.89 against 0.85 ms -- the smaller CTAs pay off only on long queues)
            for (int a2 = ag + 1; a2 <= 4; ++a2) {
                const int x2 = std::min(c->MP / 4, 3);
                if (ap % a2 == 0 && ap / a2 + x2 + 2 <= 10 && dos_sweep_ffma_angles_per_warp(ap, c->L, a2) == a2) { ag = a2; nx = x2; break; }
            }
    }
    int grid = 0;
    cudaError_t e = dos_sweep_ffma_grid(c->L, ag, nx, ap, c->n_mat, c->n_items * as, c->two_per_sm, &grid);
    if (e != cudaSuccess) return e;
    c->asplit = as; c->ag = ag; c->n_grp = ap / ag; c->n_aux = nx; c->grid = grid; c->umma = false;
    return cudaSuccess;
}

// Default angle split: one CTA per (octant, tile). Spreading an octant's angles over 2 or more CTAs (option
// "sweep_angle_split") shortens a step on meshes of a few tiles but replicates the moment staging and the
// reductions; measured on config 2 it is a wash, so it stays an option.
static int default_asplit(int per_oct, int n_tiles_items)
{
    (void)per_oct; (void)n_tiles_items;
    return 1;
}

extern "C" dos_status dos_workspace_bytes(const dos_mesh *mesh, const dos_xs *xs, const dos_quadrature *quad,
                                          int32_t P_L, int32_t n_batch, size_t *bytes_out)
{
    if (!bytes_out) return fail(nullptr, DOS_ERR_INVALID_ARG, "bytes_out is null");
    dos_status s = check_inputs(mesh, xs, quad, P_L);
    if (s != DOS_OK) return s;
    if (n_batch < 1) return fail(nullptr, DOS_ERR_INVALID_ARG, "n_batch must be >= 1");
    if (n_batch > 64) return fail(nullptr, DOS_ERR_UNSUPPORTED, "n_batch > 64");
    *bytes_out = make_layout(mesh, xs->n_mat, xs->n_group, xs->n_leg, P_L, quad->n_ang, n_batch).total;
    return DOS_OK;
}

extern "C" dos_status dos_create(dos_ctx **out, const dos_mesh *mesh, const uint8_t *d_material_ids,
                                 const dos_xs *xs, const dos_quadrature *quad, int32_t P_L, void *d_workspace,
                                 size_t workspace_bytes, void *cuda_stream)
{
    if (!out) return fail(nullptr, DOS_ERR_INVALID_ARG, "out is null");
    *out = nullptr;
    dos_status s = check_inputs(mesh, xs, quad, P_L);
    if (s != DOS_OK) return s;
    if (!d_material_ids || !d_workspace) return fail(nullptr, DOS_ERR_INVALID_ARG, "null device pointer");
    if (((uintptr_t)d_workspace) & 255) return fail(nullptr, DOS_ERR_INVALID_ARG, "workspace not 256-byte aligned");
    const int G = xs->n_group, n_mat = xs->n_mat, n_leg = xs->n_leg, L = P_L, n_ang = quad->n_ang, per = n_ang / 8;
    const int M = (L + 1) * (L + 1), MP = dos_mpad(L);
    // ---- table checks ----
    for (int i = 0; i < n_mat * G; ++i)
        if (!(xs->sigma_t[i] > 0.f)) return fail(nullptr, DOS_ERR_INVALID_ARG, "sigma_t must be > 0");
    for (int m = 0; m < n_mat; ++m)
        for (int l = 0; l <= n_leg; ++l)
            for (int gf = 0; gf < G; ++gf)
                for (int gt = 0; gt < gf; ++gt)
                    if (xs->sigma_s[(((size_t)m * (n_leg + 1) + l) * G + gf) * G + gt] != 0.f)
                        return fail(nullptr, DOS_ERR_INVALID_ARG, "sigma_s has upscatter (to < from) entries");
    double wsum = 0.0;
    for (int n = 0; n < n_ang; ++n) wsum += quad->w[n];
    if (std::fabs(wsum - 1.0) > 1e-5) return fail(nullptr, DOS_ERR_INVALID_ARG, "quadrature weights must sum to 1");
    for (int o = 0; o < 8; ++o)
        for (int t = 0; t < per; ++t) {
            const int n = o * per + t;
            const float ex = (o & 1) ? -quad->mu[t] : quad->mu[t], ey = (o & 2) ? -quad->eta[t] : quad->eta[t],
                        ez = (o & 4) ? -quad->xi[t] : quad->xi[t];
            if (!(quad->mu[t] > 0.f && quad->eta[t] > 0.f && quad->xi[t] > 0.f) || quad->mu[n] != ex ||
                quad->eta[n] != ey || quad->xi[n] != ez || quad->w[n] != quad->w[t])
                return fail(nullptr, DOS_ERR_INVALID_ARG, "quadrature is not octant-major / octant-symmetric");
        }
    // the number of position slots is what the workspace was sized for (dos_workspace_bytes' n_batch): the largest count
    // whose layout fits; with more than one slot it also holds the buffers of the summed-source mode
    int n_slots = 0;
    for (int n = 1; n <= 64 && make_layout(mesh, n_mat, G, n_leg, L, n_ang, n).total <= workspace_bytes; ++n) n_slots = n;
    if (n_slots < 1) return fail(nullptr, DOS_ERR_SHAPE, "workspace too small");
    const Layout lay = make_layout(mesh, n_mat, G, n_leg, L, n_ang, n_slots);
    const bool can_sum = n_slots > 1;

    dos_ctx *c = new (std::nothrow) dos_ctx();
    if (!c) return fail(nullptr, DOS_ERR_NOMEM, "out of host memory");
    c->mesh = *mesh;
    c->n_mat = n_mat; c->G = G; c->n_leg = n_leg; c->L = L; c->M = M; c->MP = MP; c->n_ang = n_ang; c->per_oct = per;
    c->ntj = (mesh->ny + DOS_TJ - 1) / DOS_TJ;
    c->ntk = (mesh->nz + DOS_TK - 1) / DOS_TK;
    c->n_items = 8 * c->ntj * c->ntk;
    c->n_items_u = 2 * c->ntj * c->ntk;
    c->can_sum = can_sum; c->summed = false;
    c->contraction_pref = 0;
    c->ag_pref = c->aux_pref = 0;
    c->asplit = default_asplit(per, c->n_items);
    c->chunk = 2;
    c->two_per_sm = 1;
    c->ll_pref = 1; c->epoch = 0;
    c->umma = false;
    c->grid = c->grid_u = 0;
    c->mat_checked = false;
    c->refl = 0;
    c->n_slots = n_slots; c->active = 0;
    c->srcs.resize(n_slots);
    c->nv = (size_t)mesh->nx * mesh->ny * mesh->nz;
    c->stream = (cudaStream_t)cuda_stream;
    c->d_mat = d_material_ids;
    c->ws = (char *)d_workspace;
    c->lay = lay;
    c->state = 0;
    c->have_dose_acc = false;
    c->profile = false; c->prof_open = false;
    c->acc_ms[0] = c->acc_ms[1] = 0.0;
    c->acc_n[0] = c->acc_n[1] = 0;
    c->launches = 0;

    // ---- host tables ----
    std::vector<float> sig_t_gm((size_t)G * n_mat);
    for (int m = 0; m < n_mat; ++m)
        for (int g = 0; g < G; ++g) sig_t_gm[(size_t)g * n_mat + m] = xs->sigma_t[(size_t)m * G + g];
    c->band_lo.assign(G, 0);
    for (int g = 0; g < G; ++g) {
        int lo = g;
        for (int gp = g - 1; gp >= 0; --gp)
            for (int m = 0; m < n_mat; ++m)
                for (int l = 0; l <= L; ++l)
                    if (xs->sigma_s[(((size_t)m * (n_leg + 1) + l) * G + gp) * G + g] != 0.f) lo = gp;
        c->band_lo[g] = lo;
    }
    std::vector<float> m2d((size_t)n_ang * MP, 0.f), d2m((size_t)n_ang * MP, 0.f), cdd((size_t)per * 4);
    double y[64];
    for (int n = 0; n < n_ang; ++n) {
        host_ylm((double)quad->mu[n], (double)quad->eta[n], (double)quad->xi[n], L, y);
        for (int l = 0; l <= L; ++l)
            for (int mm = -l; mm <= l; ++mm) {
                const int lm = l * (l + 1) + mm;
                m2d[(size_t)n * MP + lm] = (float)((2.0 * l + 1.0) * y[lm]);
                d2m[(size_t)n * MP + lm] = (float)((double)quad->w[n] * y[lm]);
            }
    }
    for (int t = 0; t < per; ++t) {
        const double cx = 2.0 * std::fabs((double)quad->mu[t]) / mesh->dx, cy = 2.0 * std::fabs((double)quad->eta[t]) / mesh->dy,
                     cz = 2.0 * std::fabs((double)quad->xi[t]) / mesh->dz;
        cdd[t * 4 + 0] = (float)cx; cdd[t * 4 + 1] = (float)cy; cdd[t * 4 + 2] = (float)cz;
        cdd[t * 4 + 3] = (float)(cx + cy + cz);
    }
    // work items, tile-diagonal major: every item's upwind tiles (tj-1,tk), (tj,tk-1) come earlier.
    // FFMA sweep: (octant, tile); tensor-memory sweep: (octant quad, tile)
    std::vector<int> items, items_u;
    items.reserve(c->n_items);
    items_u.reserve(c->n_items_u);
    for (int d = 0; d <= c->ntj + c->ntk - 2; ++d)
        for (int tj = 0; tj < c->ntj; ++tj) {
            const int tk = d - tj;
            if (tk < 0 || tk >= c->ntk) continue;
            for (int o = 0; o < 8; ++o) items.push_back(o | (tj << 3) | (tk << 17));
            for (int qd = 0; qd < 2; ++qd) items_u.push_back(qd | (tj << 3) | (tk << 17));
        }
    // Tensor-memory sweep tables. Y_lm of a direction mirrored into octant o is +-Y_lm of the octant-0 direction, the
    // sign depending on (l, m) and the mirror only: signs[o][lm]. The UMMA B operands hold octant 0's coefficients,
    // split into TF32 hi + lo, in the no-swizzle K-major core-matrix layout (8 rows x 16 bytes).
    const int KP = (MP + 7) & ~7, NCH = KP / 4, A8 = (per + 7) & ~7, NAP = (per + 15) & ~15, NMP = (MP + 15) & ~15;
    std::vector<unsigned> signs((size_t)8 * MP, 0u);
    std::vector<float> bm2d((size_t)2 * NAP * KP, 0.f), bd2m((size_t)2 * NMP * A8, 0.f);
    bool umma_ok = dos_sweep_umma_supported(per, L) != 0;
    for (int o = 0; o < 8 && umma_ok; ++o)
        for (int lm = 0; lm < M; ++lm) {
            int tbest = 0;
            for (int t = 1; t < per; ++t)
                if (std::fabs(m2d[(size_t)t * MP + lm]) > std::fabs(m2d[(size_t)tbest * MP + lm])) tbest = t;
            const bool neg = (m2d[((size_t)o * per + tbest) * MP + lm] < 0.f) != (m2d[(size_t)tbest * MP + lm] < 0.f);
            signs[(size_t)o * MP + lm] = neg ? 0x80000000u : 0u;
            for (int t = 0; t < per; ++t) {       // the mirror relation must hold exactly, for both tables
                const float sg = neg ? -1.f : 1.f;
                if (m2d[((size_t)o * per + t) * MP + lm] != sg * m2d[(size_t)t * MP + lm] ||
                    d2m[((size_t)o * per + t) * MP + lm] != sg * d2m[(size_t)t * MP + lm]) umma_ok = false;
            }
        }
    auto tf32 = [](float x) {
        unsigned b; std::memcpy(&b, &x, 4);
        b = (b + 0x1000u) & 0xffffe000u;
        float r; std::memcpy(&r, &b, 4);
        return r;
    };
    for (int n = 0; n < per; ++n)
        for (int k = 0; k < MP; ++k) {
            const size_t im = ((size_t)(n / 8) * NCH + k / 4) * 32 + (n % 8) * 4 + (k % 4);              // (angle n, moment k)
            const float vm = m2d[(size_t)n * MP + k], hm = tf32(vm);
            bm2d[im] = hm; bm2d[(size_t)NAP * KP + im] = tf32(vm - hm);
            const size_t id = ((size_t)(k / 8) * (A8 / 4) + n / 4) * 32 + (k % 8) * 4 + (n % 4);         // (moment k, angle n)
            const float vd = d2m[(size_t)n * MP + k], hd = tf32(vd);
            bd2m[id] = hd; bd2m[(size_t)NMP * A8 + id] = tf32(vd - hd);
        }
    c->umma_ok = umma_ok;

    auto up = [&](size_t off, const void *src, size_t bytes) {
        return cudaMemcpyAsync(c->ws + off, src, bytes, cudaMemcpyHostToDevice, c->stream);
    };
    cudaError_t e = cudaSuccess;
    if (e == cudaSuccess) e = up(lay.sig_t, sig_t_gm.data(), sizeof(float) * sig_t_gm.size());
    if (e == cudaSuccess) e = up(lay.sig_s, xs->sigma_s, sizeof(float) * (size_t)n_mat * (n_leg + 1) * G * G);
    if (e == cudaSuccess) e = up(lay.kerma, xs->kerma, sizeof(float) * n_mat * G);
    if (e == cudaSuccess) e = up(lay.m2d, m2d.data(), sizeof(float) * m2d.size());
    if (e == cudaSuccess) e = up(lay.d2m, d2m.data(), sizeof(float) * d2m.size());
    if (e == cudaSuccess) e = up(lay.cdd, cdd.data(), sizeof(float) * cdd.size());
    c->h_cdd = cdd;
    if (e == cudaSuccess) e = up(lay.items, items.data(), sizeof(int) * items.size());
    if (e == cudaSuccess) e = up(lay.items_u, items_u.data(), sizeof(int) * items_u.size());
    if (e == cudaSuccess) e = up(lay.bm2d, bm2d.data(), sizeof(float) * bm2d.size());
    if (e == cudaSuccess) e = up(lay.bd2m, bd2m.data(), sizeof(float) * bd2m.size());
    if (e == cudaSuccess) e = up(lay.signs, signs.data(), sizeof(unsigned) * signs.size());
    if (e == cudaSuccess) e = cudaMemsetAsync(c->ws + lay.errflag, 0, sizeof(int) * 4, c->stream);
    // the whole grid is checked once, here (dos.h: ids < n_mat); every kernel also clamps the id it indexes with
    if (e == cudaSuccess) e = dos_launch_validate_material(c->nv, c->d_mat, n_mat, (int *)(c->ws + lay.errflag), c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);   // host vectors go out of scope
    if (e == cudaSuccess) e = configure_sweep(c);
    if (e != cudaSuccess) {
        std::string msg = std::string("dos_create: ") + cudaGetErrorString(e);
        delete c;
        return fail(nullptr, DOS_ERR_CUDA, msg);
    }
    *out = c;
    return DOS_OK;
}

static MeshDev mesh_dev(const dos_mesh &m)
{
    MeshDev d;
    d.nx = m.nx; d.ny = m.ny; d.nz = m.nz;
    d.dx = m.dx; d.dy = m.dy; d.dz = m.dz;
    d.x0 = m.x0; d.y0 = m.y0; d.z0 = m.z0;
    return d;
}

static SourceDev source_dev(const dos_source &s)
{
    SourceDev d;
    for (int i = 0; i < 3; ++i) { d.pos[i] = s.pos[i]; d.axis[i] = s.axis[i]; d.up[i] = s.up[i]; }
    d.side[0] = s.axis[1] * s.up[2] - s.axis[2] * s.up[1];
    d.side[1] = s.axis[2] * s.up[0] - s.axis[0] * s.up[2];
    d.side[2] = s.axis[0] * s.up[1] - s.axis[1] * s.up[0];
    d.tan_fan = s.tan_half_fan; d.tan_cone = s.tan_half_cone; d.isotropic = s.isotropic;
    return d;
}

// optional CUDA-event bracket around one launch (option "profile")
static void prof_begin(dos_ctx *c, int kind)
{
    if (!c->profile) return;
    cudaEvent_t e[2];
    for (int i = 0; i < 2; ++i) {
        if (!c->ev_pool.empty()) { e[i] = c->ev_pool.back(); c->ev_pool.pop_back(); }
        else if (cudaEventCreate(&e[i]) != cudaSuccess) { c->prof_open = false; return; }
    }
    c->ev.push_back(e[0]); c->ev.push_back(e[1]); c->ev_kind.push_back(kind);
    c->prof_open = true;
    cudaEventRecord(e[0], c->stream);
}
static void prof_end(dos_ctx *c)
{
    if (!c->profile || !c->prof_open) return;
    cudaEventRecord(c->ev.back(), c->stream);
    c->prof_open = false;
}
static void prof_collect(dos_ctx *c)
{
    for (size_t i = 0; i < c->ev_kind.size(); ++i) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, c->ev[2 * i], c->ev[2 * i + 1]) == cudaSuccess) {
            c->acc_ms[c->ev_kind[i]] += ms;
            c->acc_n[c->ev_kind[i]] += 1;
        }
        c->ev_pool.push_back(c->ev[2 * i]);
        c->ev_pool.push_back(c->ev[2 * i + 1]);
    }
    c->ev.clear();
    c->ev_kind.clear();
}

extern "C" dos_status dos_set_material_host(dos_ctx *c, const uint8_t *h_material_ids)
{
    if (!c || !h_material_ids) return fail(c, DOS_ERR_INVALID_ARG, "null argument");
    // The copy is enqueued; with pageable memory the runtime stages it before returning, with pinned memory the
    // caller's buffer must stay untouched until the stream reaches this point (dos.h).
    CUDA_TRY(c, cudaMemcpyAsync(c->ws + c->lay.mat, h_material_ids, c->nv, cudaMemcpyHostToDevice, c->stream));
    c->d_mat = (const uint8_t *)(c->ws + c->lay.mat);
    // a new grid: the "bad material id" flag starts afresh and the grid is checked again
    CUDA_TRY(c, cudaMemsetAsync(c->ws + c->lay.errflag, 0, sizeof(int), c->stream));
    CUDA_TRY(c, dos_launch_validate_material(c->nv, c->d_mat, c->n_mat, (int *)(c->ws + c->lay.errflag), c->stream));
    c->launches += 1;
    c->state = 0;
    return DOS_OK;
}

// mode 0: single source; 1: first source of a sum; 2: further source of a sum
static dos_status uncollided_impl(dos_ctx *c, const dos_source *source, const float *spectrum, float *d_phi_u_out, int mode, int slot = 0)
{
    if (!c || !source || !spectrum) return fail(c, DOS_ERR_INVALID_ARG, "null argument");
    if (mode && !c->can_sum) return fail(c, DOS_ERR_STATE, "the workspace was not sized for the summed-source mode (dos_workspace_bytes with n_batch > 1)");
    if (mode == 2 && !(c->summed && c->state >= 1)) return fail(c, DOS_ERR_STATE, "dos_uncollided_sum(first = 0) without a first source");
    auto dot = [](const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; };
    if (!source->isotropic) {
        if (std::fabs(dot(source->axis, source->axis) - 1.0) > 1e-9 || std::fabs(dot(source->up, source->up) - 1.0) > 1e-9 ||
            std::fabs(dot(source->axis, source->up)) > 1e-9)
            return fail(c, DOS_ERR_INVALID_ARG, "axis and up must be orthonormal");
        if (!(source->tan_half_fan >= 0.0) || !(source->tan_half_cone >= 0.0))
            return fail(c, DOS_ERR_INVALID_ARG, "collimation tangents must be >= 0");
    }
    // a source closer than 1e-9 cm to a voxel centre has no defined direction (1/r^2 singular)
    {
        const dos_mesh &m = c->mesh;
        const double fx = (source->pos[0] - m.x0) / m.dx - 0.5, fy = (source->pos[1] - m.y0) / m.dy - 0.5,
                     fz = (source->pos[2] - m.z0) / m.dz - 0.5;
        const double rx = std::nearbyint(fx), ry = std::nearbyint(fy), rz = std::nearbyint(fz);
        if (rx >= 0 && rx < m.nx && ry >= 0 && ry < m.ny && rz >= 0 && rz < m.nz) {
            const double ex = (fx - rx) * m.dx, ey = (fy - ry) * m.dy, ez = (fz - rz) * m.dz;
            if (std::sqrt(ex * ex + ey * ey + ez * ez) < 1e-9)
                return fail(c, DOS_ERR_INVALID_ARG, "source coincides with a voxel centre");
        }
    }
    SpectrumDev sp;                                  // travels in the kernel's parameters: nothing to copy, nothing to wait for
    for (int g = 0; g < DOS_MAX_G; ++g) sp.s[g] = 0.0;
    for (int g = 0; g < c->G; ++g) {
        if (!(spectrum[g] >= 0.f)) return fail(c, DOS_ERR_INVALID_ARG, "spectrum must be >= 0");
        sp.s[g] = (double)spectrum[g];
    }
    c->srcs[slot] = *source;
    float *phi_u = (float *)(c->ws + c->lay.phi_u + (size_t)slot * c->lay.slot);
    prof_begin(c, 1);
    CUDA_TRY(c, dos_launch_raytrace(mesh_dev(c->mesh), source_dev(*source), c->d_mat, c->n_mat, c->G,
                                    (const float *)(c->ws + c->lay.sig_t), sp,
                                    phi_u, (int *)(c->ws + c->lay.errflag), c->stream));
    prof_end(c);
    c->launches += 1;
    if (mode) {
        CUDA_TRY(c, dos_launch_um_accumulate(mesh_dev(c->mesh), source_dev(*source), c->G, c->L, mode == 1, phi_u,
                                             (float *)(c->ws + c->lay.um), (float *)(c->ws + c->lay.phi_u_sum), c->stream));
        c->launches += 1;
    }
    c->summed = mode != 0;
    if (d_phi_u_out)
        CUDA_TRY(c, cudaMemcpyAsync(d_phi_u_out, phi_u, sizeof(float) * c->G * c->nv, cudaMemcpyDeviceToDevice, c->stream));
    c->active = slot + 1;
    c->state = 1;
    return DOS_OK;
}

extern "C" dos_status dos_uncollided_batch(dos_ctx *c, int32_t n_sources, const dos_source *sources, const float *spectrum,
                                           float *d_phi_u_out)
{
    if (!c || !sources) return fail(c, DOS_ERR_INVALID_ARG, "null argument");
    if (n_sources < 1 || n_sources > c->n_slots)
        return fail(c, n_sources < 1 ? DOS_ERR_INVALID_ARG : DOS_ERR_STATE,
                    "dos_uncollided_batch: the workspace was sized for fewer source positions (dos_workspace_bytes' n_batch)");
    for (int b = 0; b < n_sources; ++b) {
        dos_status st = uncollided_impl(c, &sources[b], spectrum, d_phi_u_out ? d_phi_u_out + (size_t)b * c->G * c->nv : nullptr, 0, b);
        if (st != DOS_OK) { c->state = 0; c->active = 0; return st; }
    }
    return DOS_OK;
}

extern "C" dos_status dos_uncollided(dos_ctx *c, const dos_source *source, const float *spectrum, float *d_phi_u_out)
{
    return uncollided_impl(c, source, spectrum, d_phi_u_out, 0);
}

extern "C" dos_status dos_uncollided_sum(dos_ctx *c, const dos_source *source, const float *spectrum, int32_t first,
                                         float *d_phi_u_out)
{
    return uncollided_impl(c, source, spectrum, d_phi_u_out, first ? 1 : 2);
}

extern "C" dos_status dos_uncollided_total(dos_ctx *c, float *d_phi_u_out)
{
    if (!c || !d_phi_u_out) return fail(c, DOS_ERR_INVALID_ARG, "null argument");
    if (c->state < 1) return fail(c, DOS_ERR_STATE, "dos_uncollided_total before dos_uncollided");
    const float *src = (const float *)(c->ws + (c->summed ? c->lay.phi_u_sum : c->lay.phi_u));
    CUDA_TRY(c, cudaMemcpyAsync(d_phi_u_out, src, sizeof(float) * c->G * c->nv, cudaMemcpyDeviceToDevice, c->stream));
    return DOS_OK;
}

// n_iter sweeps in every group (tol < 0), or per group until max|phi00 - phi00_old| <= tol max|phi00| with at most
// n_iter sweeps (tol >= 0; one 8-byte device-to-host read per sweep); h_iters (may be null) [G] receives the counts.
static dos_status solve_impl(dos_ctx *c, int32_t n_iter, float tol, int32_t *h_iters)
{
    if (!c) return fail(c, DOS_ERR_INVALID_ARG, "null context");
    if (c->state < 1) return fail(c, DOS_ERR_STATE, "dos_solve before dos_uncollided");
    if (n_iter < 1) return fail(c, DOS_ERR_INVALID_ARG, "n_iter must be >= 1");
    if (c->refl && !c->umma) return fail(c, DOS_ERR_UNSUPPORTED, "reflective boundaries need the tensor-memory sweep");
    if (tol >= 0.f && c->active > 1) return fail(c, DOS_ERR_UNSUPPORTED, "dos_solve_tol on a position batch");
    const int nb = c->active;                     // problems swept together (dos_uncollided_batch), 1 otherwise
    const size_t slot = c->lay.slot;
    const size_t nvm = c->nv * c->MP;
    float *phi_u = (float *)(c->ws + c->lay.phi_u), *phi_all = (float *)(c->ws + c->lay.phi_all);
    float *qfix = (float *)(c->ws + c->lay.qfix), *q = (float *)(c->ws + c->lay.q);
    const float *sig_s = (const float *)(c->ws + c->lay.sig_s);
    int *done = (int *)(c->ws + c->lay.done), *queue = (int *)(c->ws + c->lay.queue);
    const MeshDev md = mesh_dev(c->mesh);
    Sweep2Args a;                       // FFMA sweep
    a.nx = c->mesh.nx; a.ny = c->mesh.ny; a.nz = c->mesh.nz; a.ntj = c->ntj; a.ntk = c->ntk;
    a.per_oct = c->per_oct / c->asplit; a.per_oct_full = c->per_oct; a.a_split = c->asplit;
    a.n_items = c->n_items * c->asplit * nb; a.n_batch = nb; a.slot_stride = slot; a.n_warps = c->n_grp; a.n_aux = c->n_aux; a.chunk = c->chunk; a.n_mat = c->n_mat;
    a.items = (const int *)(c->ws + c->lay.items); a.Q = q; a.mat = c->d_mat;
    a.m2d = (const float *)(c->ws + c->lay.m2d); a.d2m = (const float *)(c->ws + c->lay.d2m);
    a.cdd = (const float *)(c->ws + c->lay.cdd);
    a.fy = (float *)(c->ws + c->lay.fy); a.fz = (float *)(c->ws + c->lay.fz); a.done = done; a.queue = queue;
    a.abort_flag = (int *)(c->ws + c->lay.errflag) + 1;
    SweepUArgs u;                       // tensor-memory sweep
    u.nx = a.nx; u.ny = a.ny; u.nz = a.nz; u.ntj = a.ntj; u.ntk = a.ntk; u.n_items = c->n_items_u * nb; u.n_batch = nb; u.slot_stride = slot;
    u.per_oct = c->per_oct;
    u.MP = c->MP; u.chunk = c->chunk; u.n_mat = c->n_mat;
    u.items = (const int *)(c->ws + c->lay.items_u); u.Q = q; u.mat = c->d_mat; u.cdd = a.cdd;
    for (size_t i = 0; i < sizeof(u.cddc) / sizeof(float); ++i) u.cddc[i] = i < c->h_cdd.size() ? c->h_cdd[i] : 0.f;
    u.bm2d = (const float *)(c->ws + c->lay.bm2d); u.bd2m = (const float *)(c->ws + c->lay.bd2m);
    u.signs = (const unsigned *)(c->ws + c->lay.signs);
    u.fy = a.fy; u.fz = a.fz; u.done = done; u.queue = queue; u.abort_flag = a.abort_flag;
    const int n_flags = c->umma ? c->n_items_u : c->n_items * c->asplit;
    // reflective boundaries: halves of the boundary-outflow buffers alternate between "previous sweep" and "this sweep"
    const size_t bxh = (size_t)8 * c->per_oct * c->mesh.nz * c->mesh.ny, byh = (size_t)8 * c->ntk * (c->mesh.nx + DOS_FACE_PAD) * c->per_oct * DOS_TK,
                 bzh = (size_t)8 * c->ntj * (c->mesh.nx + DOS_FACE_PAD) * c->per_oct * DOS_TJ;
    float *bx = (float *)(c->ws + c->lay.bx), *by = (float *)(c->ws + c->lay.by), *bz = (float *)(c->ws + c->lay.bz);
    float *phi00_old = tol >= 0.f ? (float *)(c->ws + c->lay.phi00_old) : nullptr;
    int *conv = (int *)(c->ws + c->lay.conv);
    u.refl = c->refl;
    int sweep_no = 0;
    for (int g = 0; g < c->G; ++g) {
        float *phi = phi_all + (size_t)g * nvm;
        for (int b = 0; b < nb; ++b) {            // the fixed source depends on the position (Y_lm of the direction from the source)
            const size_t sh = (size_t)b * slot / sizeof(float);
            CUDA_TRY(c, dos_launch_group_source(md, source_dev(c->srcs[b]), c->d_mat, c->n_mat, c->G, c->n_leg, c->L, g, c->band_lo[g], sig_s,
                                                phi_u + sh, c->summed ? (const float *)(c->ws + c->lay.um) : nullptr, phi_all + sh,
                                                qfix + sh, c->stream));
            c->launches += 1;
        }
        a.phi = u.phi = phi;
        a.sig_t = u.sig_t = (const float *)(c->ws + c->lay.sig_t) + (size_t)g * c->n_mat;
        if (c->refl) {
            // every group starts from zero boundary inflow (the lagged reflective condition of the first sweep)
            for (int b = 0; b < nb; ++b) {
                const size_t sh = (size_t)b * slot / sizeof(float);
                CUDA_TRY(c, cudaMemsetAsync(bx + sh, 0, sizeof(float) * 2 * bxh, c->stream));
                CUDA_TRY(c, cudaMemsetAsync(by + sh, 0, sizeof(float) * 2 * byh, c->stream));
                CUDA_TRY(c, cudaMemsetAsync(bz + sh, 0, sizeof(float) * 2 * bzh, c->stream));
            }
        }
        int it = 0;
        for (; it < n_iter; ++it) {
            CUDA_TRY(c, dos_launch_source_update(c->nv, c->d_mat, c->n_mat, c->G, c->n_leg, c->L, g, sig_s, qfix, phi, q, it == 0,
                                                 done, n_flags, queue, phi00_old, nb, slot, c->stream));
            const int cur = sweep_no & 1, prv = cur ^ 1;
            u.bx_in = bx + prv * bxh; u.bx_out = bx + cur * bxh;
            u.by_in = by + prv * byh; u.by_out = by + cur * byh;
            u.bz_in = bz + prv * bzh; u.bz_out = bz + cur * bzh;
            ++sweep_no;
            prof_begin(c, 0);
            if (c->umma) CUDA_TRY(c, dos_launch_sweep_umma(u, c->L, c->grid_u, c->stream));
            else {
                a.ll = (c->ll_pref && ll_mesh(&c->mesh, c->per_oct) && 3 * a.per_oct <= 32) ? 1 : 0;
                if (++c->epoch == 0 || c->epoch > 0x7fffffffu) c->epoch = 1;
                a.epoch = (int)c->epoch;
                CUDA_TRY(c, dos_launch_sweep_ffma(a, c->L, c->ag, c->grid, c->two_per_sm, c->stream));
            }
            prof_end(c);
            c->launches += 2;
            if (tol >= 0.f) {
                int h[2] = {0, 0};
                CUDA_TRY(c, dos_launch_conv(c->nv, c->MP, phi, phi00_old, conv, c->stream));
                CUDA_TRY(c, cudaMemcpyAsync(h, conv, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
                CUDA_TRY(c, cudaStreamSynchronize(c->stream));
                c->launches += 1;
                float d, m;
                std::memcpy(&d, &h[0], 4); std::memcpy(&m, &h[1], 4);
                if (d <= tol * m) { ++it; break; }
            }
        }
        if (h_iters) h_iters[g] = it;
    }
    c->state = 2;
    return DOS_OK;
}

extern "C" dos_status dos_solve(dos_ctx *c, int32_t n_iter) { return solve_impl(c, n_iter, -1.f, nullptr); }

extern "C" dos_status dos_solve_tol(dos_ctx *c, float tol, int32_t max_iter, int32_t *h_iters)
{
    if (!(tol >= 0.f)) return fail(c, DOS_ERR_INVALID_ARG, "tol must be >= 0");
    return solve_impl(c, max_iter, tol, h_iters);
}

extern "C" dos_status dos_set_boundary(dos_ctx *c, int32_t reflective_faces)
{
    if (!c) return fail(c, DOS_ERR_INVALID_ARG, "null context");
    if (reflective_faces < 0 || reflective_faces > 7) return fail(c, DOS_ERR_INVALID_ARG, "reflective_faces is a 3-bit mask (x, y, z)");
    if (reflective_faces && !c->umma_ok) return fail(c, DOS_ERR_UNSUPPORTED, "reflective boundaries need the tensor-memory sweep, which has no shape for this quadrature");
    const int old = c->refl;
    c->refl = reflective_faces;
    if (configure_sweep(c) != cudaSuccess) {
        c->refl = old;
        configure_sweep(c);
        return fail(c, DOS_ERR_UNSUPPORTED, "reflective boundaries: no admissible sweep");
    }
    return DOS_OK;
}

static dos_status check_device_flags(dos_ctx *c)
{
    int h[4] = {0, 0, 0, 0};
    CUDA_TRY(c, cudaMemcpyAsync(h, c->ws + c->lay.errflag, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    if (h[0]) return fail(c, DOS_ERR_INVALID_ARG, "material id >= n_mat met on the device");
    if (h[1]) return fail(c, DOS_ERR_CUDA, "sweep watchdog fired: a face-flux hand-off never arrived; results are invalid");
    return DOS_OK;
}

extern "C" dos_status dos_check(dos_ctx *c)
{
    if (!c) return fail(c, DOS_ERR_INVALID_ARG, "null context");
    return check_device_flags(c);
}

extern "C" dos_status dos_fluence(dos_ctx *c, float *d_phi_collided, float *d_phi_total)
{
    if (!c) return fail(c, DOS_ERR_INVALID_ARG, "null context");
    if (c->state < 2) return fail(c, DOS_ERR_STATE, "dos_fluence before dos_solve");
    for (int b = 0; b < c->active; ++b) {         // a position batch fills [n_sources][G][nz][ny][nx]
        const size_t sh = (size_t)b * c->lay.slot, out = (size_t)b * c->G * c->nv;
        CUDA_TRY(c, dos_launch_fluence(c->nv, c->G, c->MP, (const float *)(c->ws + (c->summed ? c->lay.phi_u_sum : c->lay.phi_u + sh)),
                                       (const float *)(c->ws + c->lay.phi_all + sh), d_phi_collided ? d_phi_collided + out : nullptr,
                                       d_phi_total ? d_phi_total + out : nullptr, c->stream));
        c->launches += 1;
    }
    return DOS_OK;
}

extern "C" dos_status dos_dose(dos_ctx *c, float *d_dose, int32_t accumulate)
{
    if (!c || !d_dose) return fail(c, DOS_ERR_INVALID_ARG, "null argument");
    if (c->state < 2) return fail(c, DOS_ERR_STATE, "dos_dose before dos_solve");
    for (int b = 0; b < c->active; ++b) {         // a position batch: the doses of its positions are summed (a9)
        const size_t sh = (size_t)b * c->lay.slot;
        CUDA_TRY(c, dos_launch_dose(c->nv, c->d_mat, c->n_mat, c->G, c->MP, (const float *)(c->ws + c->lay.kerma),
                                    (const float *)(c->ws + (c->summed ? c->lay.phi_u_sum : c->lay.phi_u + sh)),
                                    (const float *)(c->ws + c->lay.phi_all + sh), d_dose, accumulate || b > 0, c->stream));
        c->launches += 1;
    }
    return DOS_OK;
}

extern "C" dos_status dos_dose_host(dos_ctx *c, float *h_dose, int32_t accumulate)
{
    if (!c || !h_dose) return fail(c, DOS_ERR_INVALID_ARG, "null argument");
    float *acc = (float *)(c->ws + c->lay.dose_acc);
    dos_status s = dos_dose(c, acc, accumulate && c->have_dose_acc);
    if (s != DOS_OK) return s;
    c->have_dose_acc = true;
    CUDA_TRY(c, cudaMemcpyAsync(h_dose, acc, sizeof(float) * c->nv, cudaMemcpyDeviceToHost, c->stream));
    return check_device_flags(c);
}

extern "C" dos_status dos_set_option(dos_ctx *c, const char *name, int64_t value)
{
    if (!c || !name) return fail(c, DOS_ERR_INVALID_ARG, "null argument");
    // sweep-shape options: set, re-configure, and on failure restore what was in force
    const int old_ag = c->ag_pref, old_aux = c->aux_pref, old_as = c->asplit, old_pref = c->contraction_pref, old_two = c->two_per_sm;
    bool reshape = false;
    if (!strcmp(name, "sweep_chunk")) {
        if (value < 1) return fail(c, DOS_ERR_INVALID_ARG, "sweep_chunk must be >= 1");
        c->chunk = (int)value;
    } else if (!strcmp(name, "sweep_angles_per_warp")) {
        if (value < 0 || value > 16) return fail(c, DOS_ERR_INVALID_ARG, "sweep_angles_per_warp out of range");
        c->ag_pref = (int)value; reshape = true;
    } else if (!strcmp(name, "sweep_aux_warps")) {
        if (value < 0 || value > 16) return fail(c, DOS_ERR_INVALID_ARG, "sweep_aux_warps out of range");
        c->aux_pref = (int)value; reshape = true;
    } else if (!strcmp(name, "sweep_angle_split")) {
        if (value < 0 || value > 8 || (value > 0 && c->per_oct % value))
            return fail(c, DOS_ERR_INVALID_ARG, "sweep_angle_split must divide the angles per octant (<= 8)");
        c->asplit = value > 0 ? (int)value : default_asplit(c->per_oct, c->n_items); reshape = true;
    } else if (!strcmp(name, "sweep_contraction")) {
        if (value < 0 || value > 2) return fail(c, DOS_ERR_INVALID_ARG, "sweep_contraction must be 0 (auto), 1 (FFMA) or 2 (tensor memory)");
        c->contraction_pref = (int)value; reshape = true;
    } else if (!strcmp(name, "sweep_two_per_sm")) {
        if (value < 0 || value > 2) return fail(c, DOS_ERR_INVALID_ARG, "sweep_two_per_sm must be 0, 1 or 2");
        c->two_per_sm = (int)value; reshape = true;
    } else if (!strcmp(name, "sweep_ll")) {
        if (value < 0 || value > 1) return fail(c, DOS_ERR_INVALID_ARG, "sweep_ll must be 0 or 1");
        c->ll_pref = (int)value; reshape = true;      // (re-zeroes the pair buffers)
    } else if (!strcmp(name, "profile")) {
        c->profile = value != 0;
    } else if (!strcmp(name, "sweep_grid")) {
        if (value < 1) return fail(c, DOS_ERR_INVALID_ARG, "sweep_grid must be >= 1");
        c->grid = (int)(value < c->n_items * c->asplit ? value : c->n_items * c->asplit);
        c->grid_u = (int)(value < c->n_items_u ? value : c->n_items_u);
    } else {
        return fail(c, DOS_ERR_INVALID_ARG, std::string("unknown option ") + name);
    }
    if (reshape && configure_sweep(c) != cudaSuccess) {
        c->ag_pref = old_ag; c->aux_pref = old_aux; c->asplit = old_as; c->contraction_pref = old_pref; c->two_per_sm = old_two;
        configure_sweep(c);
        return fail(c, DOS_ERR_INVALID_ARG, std::string(name) + ": not admissible for this quadrature / sweep shape");
    }
    return DOS_OK;
}

extern "C" dos_status dos_profile(dos_ctx *c, dos_profile_t *out)
{
    if (!c || !out) return fail(c, DOS_ERR_INVALID_ARG, "null argument");
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    prof_collect(c);
    out->sweep_ms = c->acc_ms[0]; out->sweep_launches = c->acc_n[0];
    out->raytrace_ms = c->acc_ms[1]; out->raytrace_launches = c->acc_n[1];
    out->kernel_launches = c->launches;
    return DOS_OK;
}

extern "C" dos_status dos_profile_reset(dos_ctx *c)
{
    if (!c) return fail(c, DOS_ERR_INVALID_ARG, "null context");
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    prof_collect(c);
    c->acc_ms[0] = c->acc_ms[1] = 0.0;
    c->acc_n[0] = c->acc_n[1] = 0;
    c->launches = 0;
    return DOS_OK;
}

extern "C" void dos_destroy(dos_ctx *c)
{
    if (!c) return;
    cudaStreamSynchronize(c->stream);
    prof_collect(c);
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    delete c;
}

extern "C" const char *dos_last_error(const dos_ctx *c) { return c ? c->err.c_str() : g_err.c_str(); }
