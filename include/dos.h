/* dos.h -- C ABI of the discrete-ordinates CT dose hot path on one B200 (sm_100a).
 *
 * Method: Norris & Liu, "Photon Fluence and Dose Estimation in CT using a Discrete Ordinates
 * Boltzmann Solver", arXiv 1811.12391 (text: /root/reference/PAPER.md; cited below as PAPER.md:line).
 * Readings of points the paper leaves open are R1..R18 in DESIGN.md.
 *
 * Conventions
 *   - "host" pointers are ordinary CPU memory and are COPIED during the call that takes them.
 *   - "device" pointers (prefix d_) are CUDA device memory owned by the caller (e.g. torch tensors).
 *     The library never allocates device memory: all of its state lives in the caller's workspace,
 *     which must stay alive and untouched until dos_destroy.
 *   - Every call only ENQUEUES work on the CUDA stream given to dos_create (no host sync), except
 *     dos_create itself, the *_host entry points that copy OUT (dos_dose_host), dos_check and dos_profile*, which
 *     synchronise that stream before returning. Small host arguments (source, spectrum) are passed to the kernels by
 *     value, so they may be freed as soon as the call returns.
 *   - Fields are [..][nz][ny][nx], x fastest. Group index 0 is the HIGHEST energy.
 *   - Errors: a negative dos_status, never an exception; text via dos_last_error().
 *   - Call order: dos_create -> dos_uncollided -> dos_solve -> dos_fluence / dos_dose (any order,
 *     any number of times) -> dos_uncollided (next source position) ...; out-of-order = DOS_ERR_STATE.
 */
#ifndef DOS_H_
#define DOS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dos_ctx dos_ctx; /* opaque; created by dos_create, freed by dos_destroy */

typedef enum {
    DOS_OK = 0,
    DOS_ERR_INVALID_ARG = -1, /* null pointer, non-positive size, bad table values            */
    DOS_ERR_SHAPE = -2,       /* sizes inconsistent with each other / workspace too small     */
    DOS_ERR_STATE = -3,       /* call out of order                                            */
    DOS_ERR_NOMEM = -4,       /* host allocation failed                                       */
    DOS_ERR_CUDA = -5,        /* a CUDA runtime call or an earlier kernel failed              */
    DOS_ERR_UNSUPPORTED = -6  /* valid request outside what this build implements             */
} dos_status;

/* 3-D Cartesian voxel mesh. (x0,y0,z0) = lower corner in cm; voxel (i,j,k) has its
 * centre at x0 + (i + 1/2) dx, ... */
typedef struct {
    int32_t nx, ny, nz;
    double dx, dy, dz;
    double x0, y0, z0;
} dos_mesh;

/* Multigroup macroscopic cross sections per material id and dose factors
 * (PAPER.md:47, :93). All host, all fp32.
 *   sigma_t [n_mat][G]                    1/cm, > 0
 *   sigma_s [n_mat][n_leg+1][G from][G to] Legendre moments sigma_sl^{g'->g}; entries with to < from
 *                                         (upscatter) must be 0: eq. 2's g' sum is one-sided
 *                                         (reading R1)
 *   kerma   [n_mat][G]                    dose per unit fluence; a zero row neglects dose in that
 *                                         material (air)                        */
typedef struct {
    int32_t n_mat, n_group, n_leg;
    const float *sigma_t;
    const float *sigma_s;
    const float *kerma;
} dos_xs;

/* S_N quadrature (PAPER.md:43-45 eq. 3, :79). Host fp32 arrays of length n_ang = 8 * per_octant,
 * octant-major: octant o = bit0 (mu<0) | bit1 (eta<0) | bit2 (xi<0) holds entries
 * [o*per_octant, (o+1)*per_octant), and entry t of octant o is the mirror image of entry t of
 * octant 0 with the same weight. sum(w) = 1 (reading R4). */
typedef struct {
    int32_t n_ang;
    const float *mu, *eta, *xi, *w;
} dos_quadrature;

/* Point source with rectangular-pyramid collimation ("position ... two additional
 * parameters phi and theta"; reading R8). axis, up: unit vectors, up perpendicular to axis. A voxel
 * centre c is inside the beam iff isotropic != 0, or with d = c - pos, a = d.axis > 0:
 * |d.up| <= a tan_half_cone and |d.(axis x up)| <= a tan_half_fan (boundary inclusive). */
typedef struct {
    double pos[3];
    double axis[3];
    double up[3];
    double tan_half_fan, tan_half_cone;
    int32_t isotropic;
} dos_source;

/* Bytes of device workspace dos_create needs for this problem. n_batch (1..64) = source positions that can be in flight
 * at once: dos_uncollided_batch traces up to n_batch positions and dos_solve then sweeps them together (SURVEY.md 8(f)
 * N2); each position owns its own uncollided fluence, moments of all groups, sweep source and face buffers (a "slot").
 * n_batch > 1 also adds the buffers of the summed-source mode (dos_uncollided_sum): [G][Nv][MP] + [G][Nv] floats.
 * dos_create reads the slot count back from the size of the workspace it is given. */
dos_status dos_workspace_bytes(const dos_mesh *mesh, const dos_xs *xs, const dos_quadrature *quad,
                               int32_t P_L, int32_t n_batch, size_t *bytes_out);

/* Build a context: validates and copies the host tables, precomputes the moment-to-discrete and
 * discrete-to-moment matrices ((2l+1) Y_lm(Omega_n) and w_n Y_lm(Omega_n); real Schmidt
 * semi-normalised harmonics, (P_L+1)^2 moments; readings R2, R10) and the diamond-difference
 * constants 2|Omega_d|/Delta_d, and lays out the workspace.
 *   d_material_ids  device uint8 [nz][ny][nx], values < n_mat: the whole grid is checked on the device here (and again
 *                   by dos_set_material_host); an id >= n_mat is reported by dos_check / dos_dose_host as
 *                   DOS_ERR_INVALID_ARG, and every kernel clamps the id it indexes a table with, so a bad grid gives a
 *                   flagged, wrong result, never an out-of-bounds access; caller-owned, must outlive the context
 *   P_L             scattering order used, 0 <= P_L <= min(xs->n_leg, 5)
 *   d_workspace     device, >= dos_workspace_bytes, 256-byte aligned
 *   cuda_stream     a cudaStream_t (NULL = legacy default stream)                                  */
dos_status dos_create(dos_ctx **out, const dos_mesh *mesh, const uint8_t *d_material_ids,
                      const dos_xs *xs, const dos_quadrature *quad, int32_t P_L, void *d_workspace,
                      size_t workspace_bytes, void *cuda_stream);

/* Replace the material grid from HOST memory (copied into the workspace; the context then uses that
 * copy instead of d_material_ids) and check it (as dos_create does; the bad-id flag of the previous grid is cleared).
 * Used by the end-to-end path. The copy is only enqueued: pageable memory is staged by the CUDA runtime before the
 * call returns; PINNED memory must stay untouched until the stream has passed this point. */
dos_status dos_set_material_host(dos_ctx *ctx, const uint8_t *h_material_ids);

/* Uncollided fluence by ray tracing (readings R6-R9): for every voxel centre inside
 * the beam, phi_u^g = S_g exp(-sum_cells sigma_t^g l_cell) / (4 pi r^2) with exact (Siddon) segment
 * lengths from the source to the voxel CENTRE, no attenuation outside the mesh; 0 outside the beam.
 * Accumulated and exponentiated in fp64, stored as fp32 in the workspace.
 *   spectrum        host [G], source particles per group (sum = 1 for "per source particle")
 *   d_phi_u_out     device [G][nz][ny][nx] or NULL: also copy the result there                      */
dos_status dos_uncollided(dos_ctx *ctx, const dos_source *source, const float *spectrum,
                          float *d_phi_u_out);

/* Position batch (BASELINE.json config 4: an axial scan is a set of independent problems on one mesh):
 * the uncollided fluence of n_sources positions (host array; 1 <= n_sources <= the n_batch the workspace was sized for),
 * one slot each. The following dos_solve sweeps all of them in the SAME launches -- the work queue of a sweep holds the
 * (position, octant, tile) items of every position, so that small meshes fill the SMs and the tile-wavefront tail of one
 * position overlaps the head of the next; results are those of separate solves, bit for bit up to the order of the
 * moment reductions. dos_fluence then fills [n_sources][G][nz][ny][nx], dos_dose returns the SUM of the positions' dose
 * maps (a9). d_phi_u_out: device [n_sources][G][nz][ny][nx] or NULL. */
dos_status dos_uncollided_batch(dos_ctx *ctx, int32_t n_sources, const dos_source *sources, const float *spectrum,
                                float *d_phi_u_out);

/* Summed-source mode (the cone beams of a CT scan form ONE source and
 * the S_N equations are solved once). Like dos_uncollided, but the uncollided fluence of this source is ADDED to
 * that of the sources given since the last call with first != 0: phi_u = sum_p phi_u,p, and the first-collision
 * source of the following dos_solve is sum_p Y_lm(Omega_p) sum_{g'<=g} sigma_sl^{g'->g} phi_u,p^{g'} (each position
 * with its own direction Omega_p from the source to the cell). first != 0 starts a new sum. dos_fluence and
 * dos_dose then report the summed uncollided fluence plus the one collided solution. By linearity this equals the
 * sum of the per-position solves wherever the negative-flux fixup does not fire; it is NOT config 4's
 * sum of separate solves. d_phi_u_out (device [G][nz][ny][nx], may be NULL) receives this source's own phi_u.
 * Needs a workspace sized by dos_workspace_bytes with n_batch > 1 (else DOS_ERR_STATE). */
dos_status dos_uncollided_sum(dos_ctx *ctx, const dos_source *source, const float *spectrum, int32_t first,
                              float *d_phi_u_out);

/* The uncollided fluence the context currently holds -- of the last dos_uncollided, or the running sum over the
 * positions given to dos_uncollided_sum since first != 0 -- copied to device [G][nz][ny][nx]. */
dos_status dos_uncollided_total(dos_ctx *ctx, float *d_phi_u_out);

/* The same ray trace (readings R6-R9) for callers that CANNOT ALLOCATE device memory and so have
 * no workspace to give dos_create (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): no context, no workspace, no cudaMalloc / cudaFree / allocating routine inside. The kernel's scratch
 * (its [G][n_mat] cross-section table and bad-material flag) lives in a static device array of
 * DOS_STATIC_SCRATCH_BYTES that every GPU loading the library holds until the process exits.
 *   mesh, source, spectrum   as for dos_create / dos_uncollided (host)
 *   d_material_ids           device [nz][ny][nx], caller-owned
 *   sigma_t                  host [n_mat][n_group], > 0; read before the call returns
 *   d_phi_u_out              device [n_group][nz][ny][nx], caller-owned: the result (bit-identical to dos_uncollided's)
 *   d_bad_material_out       device, one int32, or NULL: 1 if a material id >= n_mat was met inside the beam (ids are
 *                            clamped for the table look-up), else 0
 *   cuda_stream              everything is enqueued on it; nothing is synchronised
 * LIMIT: n_mat <= 16 and n_group <= 64 (the table must fit the scratch); beyond that DOS_ERR_UNSUPPORTED.
 * SHARED STATE: every call uses the same array, which keeps the last call's contents; each call rewrites its table and
 * clears the flag on its stream first. Calls that overlap on the GPU (streams without an ordering between them,
 * several host threads) RACE; calls on one stream are safe. Errors: message via dos_static_last_error (per thread). */
#define DOS_STATIC_SCRATCH_BYTES 4352
dos_status dos_uncollided_static(const dos_mesh *mesh, const uint8_t *d_material_ids, int32_t n_mat, int32_t n_group,
                                 const float *sigma_t, const dos_source *source, const float *spectrum,
                                 float *d_phi_u_out, int32_t *d_bad_material_out, void *cuda_stream);
const char *dos_static_last_error(void);

/* Collided fluence (PAPER.md:39-45 eq. 2-3, :49): for g = 0..G-1, top-down (downscatter only):
 *   Q_fix = first-collision source moments Y_lm(Omega_r) sum_{g'<=g} sigma_sl^{g'->g} phi_u^{g'}
 *           + sum_{g'<g} sigma_sl^{g'->g} phi_c^{g'}[lm]
 *   n_iter source iterations from phi = 0: Q = Q_fix + sigma_sl^{g->g} phi; phi = Sweep(Q)
 * Sweep = all N_a ordinates, diamond difference with set-to-zero fixup and rebalance (north_star;
 * readings R3, R11, R12), vacuum boundaries, fp32. No convergence test (reading R5). */
dos_status dos_solve(dos_ctx *ctx, int32_t n_iter);

/* The same with a stopping rule the paper does not state: in each group the source iteration stops
 * after the first sweep with max_c |phi00^(it) - phi00^(it-1)| <= tol * max_c |phi00^(it)|, or after max_iter sweeps.
 * h_iters (host [G], may be NULL) receives the sweeps done per group. Synchronises the stream once per sweep (one
 * 8-byte read-back), so this entry point is NOT enqueue-only. */
dos_status dos_solve_tol(dos_ctx *ctx, float tol, int32_t max_iter, int32_t *h_iters);

/* Boundary condition of the following solves. reflective_faces: bit 0 the two x faces, bit 1 y, bit 2 z; 0 (default) =
 * vacuum on all faces. A reflective face returns, in each sweep, the outflow of the mirror-image ordinate
 * of the PREVIOUS sweep of the same group (lagged; zero in a group's first sweep), which converges to the specular
 * condition; it is what the infinite-medium check of north_star (phi = Q / (sigma_t - sigma_s0)) needs on the GPU.
 * Served by the tensor-memory sweep only: DOS_ERR_UNSUPPORTED for a quadrature it has no shape for. */
dos_status dos_set_boundary(dos_ctx *ctx, int32_t reflective_faces);

/* Scalar fluence per group: collided phi_c^g = phi^g[00] and/or total phi_u^g + phi_c^g.
 * Either pointer may be NULL. device [G][nz][ny][nx] fp32. */
dos_status dos_fluence(dos_ctx *ctx, float *d_phi_collided, float *d_phi_total);

/* Dose map D(c) = sum_g kerma[m(c)][g] (phi_u^g + phi_c^g)(c). device [nz][ny][nx];
 * accumulate != 0 adds to what d_dose holds (axial scan: doses of source positions summed). */
dos_status dos_dose(dos_ctx *ctx, float *d_dose, int32_t accumulate);

/* Same as dos_dose, result copied to HOST memory [nz][ny][nx]; synchronises the stream. With
 * accumulate != 0 the device-side running sum kept in the workspace is extended and returned. */
dos_status dos_dose_host(dos_ctx *ctx, float *h_dose, int32_t accumulate);

/* Synchronises the stream and reports what the kernels flagged on the device since dos_create:
 * a material id >= n_mat (DOS_ERR_INVALID_ARG), a stuck sweep hand-off or a CUDA fault (DOS_ERR_CUDA). */
dos_status dos_check(dos_ctx *ctx);

/* Tuning / measurement knobs (all optional, all per context).
 *   "sweep_contraction"  where the sweep's moment-to-discrete / discrete-to-moment contractions run: 0 (default) the
 *                   tensor-memory sweep (tcgen05.mma kind::tf32, 3xTF32 split; dos_sweep_umma.cu) wherever the quadrature
 *                   admits it and the FFMA sweep (dos_sweep_ffma.cu) otherwise; 1 FFMA; 2 tensor memory
 *   "sweep_chunk"   steps along x between face-flux hand-off publications of neighbouring tiles (>= 1)
 *   "sweep_grid"    number of persistent sweep CTAs
 *   "sweep_angles_per_warp", "sweep_aux_warps", "sweep_angle_split", "sweep_two_per_sm"  shape of the FFMA sweep CTA
 *                   (0 = library default)
 *   "sweep_ll"      FFMA sweep on small meshes (at most 128 tiles, at most 10 angles per octant): 1 (default) tile faces
 *                   travel as (value, epoch) pairs that the downwind tile polls directly; 0 the flag protocol of large meshes
 *   "profile"       1: bracket every sweep and ray-trace launch with CUDA events (see dos_profile)  */
dos_status dos_set_option(dos_ctx *ctx, const char *name, int64_t value);

/* Accumulated device time (ms, CUDA events on the context's stream) and launch counts since the last
 * dos_profile_reset, for the two named kernels. Synchronises the stream. Needs option profile=1. */
typedef struct {
    double sweep_ms;
    int64_t sweep_launches;
    double raytrace_ms;
    int64_t raytrace_launches;
    int64_t kernel_launches; /* every kernel this library launched, all kinds */
} dos_profile_t;
dos_status dos_profile(dos_ctx *ctx, dos_profile_t *out);
dos_status dos_profile_reset(dos_ctx *ctx);

void dos_destroy(dos_ctx *ctx);

/* Text of the last error of this context ("" if none); with ctx == NULL, of the last failed
 * dos_create / dos_workspace_bytes in this thread. The pointer stays valid until the next call. */
const char *dos_last_error(const dos_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* DOS_H_ */
