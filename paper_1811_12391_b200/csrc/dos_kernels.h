// dos_kernels.h -- launchers of the streaming kernels of libdos (dos_kernels.cu).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

struct MeshDev {
    int nx, ny, nz;
    double dx, dy, dz, x0, y0, z0;
};

struct SourceDev {
    double pos[3], axis[3], up[3], side[3];
    double tan_fan, tan_cone;
    int isotropic;
};

#define DOS_MAX_G 64        // energy groups (the spectrum travels in the ray-trace kernel's parameters)
struct SpectrumDev {
    double s[DOS_MAX_G];
};

// a1: phi_u[g][cell] = S_g exp(-tau_g)/(4 pi r^2) inside the beam (fp64 inside, fp32 store).
// sig_t_gm [G][n_mat]; spectrum by value (no host buffer has to outlive the call); errflag[0] set if a material id >= n_mat is met.
cudaError_t dos_launch_raytrace(const MeshDev &m, const SourceDev &s, const uint8_t *mat, int n_mat, int G,
                                const float *sig_t_gm, const SpectrumDev &spectrum, float *phi_u, int *errflag,
                                cudaStream_t st);

// a2 + a3: Q_fix[cell][lm] = Y_lm(Omega_r) sum_{g'<=g} sig_s[m][l][g'->g] phi_u[g'] +
//                            sum_{g_lo<=g'<g} sig_s[m][l][g'->g] phi_all[g'][cell][lm]
cudaError_t dos_launch_group_source(const MeshDev &m, const SourceDev &s, const uint8_t *mat, int n_mat, int G, int n_leg,
                                    int L, int g, int g_lo, const float *sig_s, const float *phi_u,
                                    const float *um /* [G][Nv][MP] summed-source mode, else null */,
                                    const float *phi_all, float *qfix, cudaStream_t st);

// summed-source mode: U^g[lm] (+)= Y_lm(Omega_p) phi_u,p^g, phi_u_sum^g (+)= phi_u,p^g after the ray trace of position p
cudaError_t dos_launch_um_accumulate(const MeshDev &m, const SourceDev &s, int G, int L, int first, const float *phi_u_pos,
                                     float *um, float *phi_u_sum, cudaStream_t st);

// a4: Q = Q_fix + sig_s[m][l][g->g] phi (phi ignored when first != 0); phi = 0; also clears the sweep's
// flags (n_flags ints at `done`) and its queue head.
cudaError_t dos_launch_source_update(size_t nv, const uint8_t *mat, int n_mat, int G, int n_leg, int L, int g,
                                     const float *sig_s, const float *qfix, float *phi, float *q, int first,
                                     int *done, int n_flags, int *queue, float *phi00_old /* or null */, int n_batch,
                                     size_t slot_stride /* bytes between the problems of a position batch */, cudaStream_t st);
// out2[0] = max |phi00 - phi00_old|, out2[1] = max |phi00| over the cells, as float bit patterns
cudaError_t dos_launch_conv(size_t nv, int MP, const float *phi, const float *phi00_old, int *out2, cudaStream_t st);

// a8: scalar fluences and dose.
cudaError_t dos_launch_fluence(size_t nv, int G, int MP, const float *phi_u, const float *phi_all,
                               float *phi_c_out, float *phi_tot_out, cudaStream_t st);
cudaError_t dos_launch_dose(size_t nv, const uint8_t *mat, int n_mat, int G, int MP, const float *kerma,
                            const float *phi_u, const float *phi_all, float *dose, int accumulate,
                            cudaStream_t st);

// errflag[0] = 1 if any material id of the grid is >= n_mat (run once per grid)
cudaError_t dos_launch_validate_material(size_t nv, const uint8_t *mat, int n_mat, int *errflag, cudaStream_t st);
