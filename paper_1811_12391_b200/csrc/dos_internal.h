// dos_internal.h -- shared between the translation units of libdos (CUDA path only).
// Nothing here is used by, or taken from, oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define DOS_MAX_MAT 16      // material ids (ray-trace per-material path-length slots in shared memory)
#define DOS_MAX_L 5         // highest P_L
#define DOS_TJ 8            // sweep tile: lanes of a warp cover TJ x TK (j,k) columns and march along x
#define DOS_TK 4
#define DOS_SKEW (DOS_TJ + DOS_TK - 2)
#define DOS_SPIN_LIMIT (1 << 22)   // polls of an upwind flag before the sweep declares itself stuck

// number of moments (L+1)^2 padded to a multiple of 4 so that a cell's moments are whole float4s
static inline __host__ __device__ int dos_mpad(int L) { return (((L + 1) * (L + 1)) + 3) & ~3; }

// ---- dos_sweep_ffma.cu: the sweep with FFMA contractions ----
#define DOS_FACE_PAD 8      // diagonal index d = x + (lane offset) runs over [0, nx + DOS_FACE_PAD)
#define DOS_PREFETCH_Q 6    // steps between issuing the cp.async of a step's source moments and using them
#define DOS_RING_Q 8
#ifndef DOS_PREFETCH_F
#define DOS_PREFETCH_F 2    // the same for tile-inflow faces (each step of it is a step of hand-off lag per tile hop)
#endif
#ifndef DOS_POLL_NS
#define DOS_POLL_NS 64      // pause between polls of a hand-off flag / of the shared progress words
#endif
#define DOS_RING_F 4

// Arguments of one launch (all 8 octants, one energy group, one source iteration).
struct Sweep2Args {
    int nx, ny, nz;
    int ntj, ntk;            // tiles along j and k
    int n_items;             // 8 * ntj * ntk * a_split work items (octant, tile, angle part); item = tile item * a_split + part
    int per_oct;             // angles per CTA (A = angles per octant / a_split)
    int per_oct_full;        // angles per octant
    int a_split;             // CTAs (angle parts) per (octant, tile)
    int n_warps;             // compute warps per CTA (A / AG)
    int n_aux;               // aux warps per CTA (staging + D2M); the CTA has one more (service) warp
    int chunk;               // steps between flag publications
    int n_mat;
    const int *items;        // [8 * ntj * ntk] packed (octant | tj << 3 | tk << 17), dependency-safe order
    const float *Q;          // [Nv][MP] frozen source moments
    float *phi;              // [Nv][MP] accumulates w Y psi (zeroed before the launch)
    const uint8_t *mat;      // [Nv]
    const float *sig_t;      // [n_mat] total cross section of this group
    const float *m2d;        // [8][per_oct_full][MP] (2l+1) Y_lm(Omega_n)
    const float *d2m;        // [8][per_oct_full][MP] w_n Y_lm(Omega_n)
    const float *cdd;        // [per_oct_full][4] cx, cy, cz, cx+cy+cz
    float *fy;               // [n_items (by id)][nx + PAD][A][TK] y-face fluxes leaving a tile, by diagonal
    float *fz;               // [n_items (by id)][nx + PAD][A][TJ] z-face fluxes leaving a tile, by diagonal
    int *done;               // [n_items (by id)] steps finished and published
    int *queue;              // work-queue head
    int *abort_flag;         // set by the watchdog; every waiting CTA then stops waiting
    // position batch: n_batch independent problems on the same mesh / tables in one launch. Work item
    // i is tile item i / n_batch of problem i % n_batch; Q, phi, fy, fz, done of problem b sit slot_stride BYTES x b
    // behind the pointers above.
    int n_batch;
    size_t slot_stride;
    // Small meshes: flag-in-data hand-off of the tile faces. Every face value travels as an 8-byte (value, epoch) pair
    // written with one store; the downwind tile polls the pairs themselves, so a hop costs one L2 round trip instead of
    // the chain progress word -> release flag -> poll -> acquire -> allowed word -> copy. fy / fz then hold pairs (twice
    // the bytes), zeroed once; epoch (> 0) differs from launch to launch so that last sweep's pairs read as "not yet".
    int ll;
    int epoch;
};

cudaError_t dos_launch_sweep_ffma(const Sweep2Args &a, int L, int ang_per_warp, int grid, int two_per_sm, cudaStream_t s);
int dos_sweep_ffma_angles_per_warp(int per_oct, int L, int prefer);
cudaError_t dos_sweep_ffma_grid(int L, int ang_per_warp, int n_aux, int per_oct, int n_mat, int n_items, int two_per_sm, int *grid_out);
int dos_sweep_ffma_aux_warps(int per_oct, int L, int ang_per_warp, int prefer);

// ---- dos_sweep_umma.cu: the sweep on the tensor-memory path (tcgen05.mma + bulk copies + mbarrier rings) ----
// One launch = all 8 octants, one energy group, one source iteration. Work item = (octant quad, tile).
struct SweepUArgs {
    int nx, ny, nz;
    int ntj, ntk;            // tiles along j and k
    int n_items;             // 2 * ntj * ntk work items (quad, tile)
    int per_oct;             // angles per octant (A)
    int MP;                  // moments per cell, padded to a multiple of 4
    int chunk;               // steps between flag publications
    int n_mat;
    const int *items;        // [n_items] packed (quad | tj << 3 | tk << 17), dependency-safe order
    const float *Q;          // [Nv][MP] frozen source moments
    float *phi;              // [Nv][MP] accumulates w Y psi (zeroed before the launch)
    const uint8_t *mat;      // [Nv]
    const float *sig_t;      // [n_mat] total cross section of this group
    const float *cdd;        // [A][4] cx, cy, cz, cx+cy+cz
    float cddc[48 * 4];      // the same by value: the cell update reads it from the constant bank, not through the LSU
    const float *bm2d;       // UMMA B operand of the moment-to-discrete: [hi, lo][NAP/8][KP/4][8][4], (angle, lm) = (2l+1) Y_lm, octant 0
    const float *bd2m;       // UMMA B operand of the discrete-to-moment: [hi, lo][NMP/8][A8/4][8][4], (lm, angle) = w Y_lm, octant 0
    const unsigned *signs;   // [8][MP] sign bit of Y_lm(mirror_o Omega) / Y_lm(Omega)
    float *fy;               // [8 * ntj * ntk (by octant, tile)][nx + PAD][A][TK] y-face fluxes leaving a tile, by diagonal
    float *fz;               // [8 * ntj * ntk][nx + PAD][A][TJ]
    int *done;               // [2 * ntj * ntk (by quad, tile)] steps finished and published
    int *queue;              // work-queue head
    int *abort_flag;
    // reflective boundaries (lagged: the inflow of an ordinate is the outflow of its mirror image in the
    // previous sweep). refl bit 0 / 1 / 2: x / y / z faces. The boundary fluxes of sweep s live in half (s & 1):
    const float *bx_in;      // [8][A][nz][ny]   x-boundary outflow of the previous sweep (octant, angle, k, j: global indices)
    float *bx_out;           //                  ... of this sweep
    const float *by_in;      // [8][ntk][nx + PAD][A][TK]  y-boundary outflow of the previous sweep, tile-face layout (by diagonal)
    float *by_out;
    const float *bz_in;      // [8][ntj][nx + PAD][A][TJ]
    float *bz_out;
    int refl;
    // position batch: work item i is tile item i / n_batch of problem i % n_batch; Q, phi, fy, fz, done
    // and the boundary buffers of problem b sit slot_stride BYTES x b behind the pointers above.
    int n_batch;
    size_t slot_stride;
};
int dos_sweep_umma_supported(int per_oct, int L);
cudaError_t dos_sweep_umma_grid(int L, int per_oct, int n_mat, int n_items, int *grid_out);
cudaError_t dos_launch_sweep_umma(const SweepUArgs &a, int L, int grid, cudaStream_t s);
