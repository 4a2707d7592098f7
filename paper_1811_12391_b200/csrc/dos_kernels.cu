// dos_kernels.cu -- the per-voxel-parallel kernels of the hot path: uncollided ray trace (a1),
// first-collision + downscatter source (a2, a3), in-group source update (a4), fluence and dose (a8).
// Moment fields are [cell][MP] (a cell's moments are contiguous float4s, MP = (L+1)^2 padded to 4).
#include "dos_internal.h"
#include "dos_kernels.h"

namespace {

constexpr int RT_THREADS = 128;

// ------------------------------------------------------------------------------------------------
// a1. Uncollided fluence ("computable with a ray-tracing algorithm"; R6-R9).
// One thread per voxel. The ray is walked BACKWARDS, from the voxel centre towards the source, with
// exact plane-crossing parameters (Siddon): beta in [0,1] along c -> s; the next crossing on each axis
// advances by a per-axis constant in fp64 (<= 1e-13 drift over a few hundred steps). Runs of equal material are merged:
// the length of a run is (beta_end - beta_start) r, added to that material's slot; the n_mat x G
// contraction with sigma_t and the exponential happen once per voxel, all in fp64.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(RT_THREADS) raytrace_kernel(MeshDev m, SourceDev s, const uint8_t *__restrict__ mat,
                                                              int n_mat, int G, const float *__restrict__ sig_t_gm,
                                                              const SpectrumDev spectrum,
                                                              float *__restrict__ phi_u, int *errflag)
{
    __shared__ double s_len[DOS_MAX_MAT][RT_THREADS];
    const size_t nv = (size_t)m.nx * m.ny * m.nz;
    // No thread leaves early: the lanes of a warp finish their walks at different steps, and without a convergence
    // point behind the walk the per-group epilogue (fp64 exp) ran once per LANE (ncu: 117 SASS instructions at one
    // active thread each, 77 % of the kernel's instructions). All 32 lanes meet at the __syncwarp() below.
    const size_t cell_raw = (size_t)blockIdx.x * RT_THREADS + threadIdx.x;
    const bool in_mesh = cell_raw < nv;
    const size_t cell = in_mesh ? cell_raw : nv - 1;
    const int i = (int)(cell % m.nx), j = (int)((cell / m.nx) % m.ny), k = (int)(cell / ((size_t)m.nx * m.ny));
    // voxel centre and d = c - s with the roundings of plain (unfused) double arithmetic
    const double cx = __dadd_rn(m.x0, __dmul_rn((double)i + 0.5, m.dx));
    const double cy = __dadd_rn(m.y0, __dmul_rn((double)j + 0.5, m.dy));
    const double cz = __dadd_rn(m.z0, __dmul_rn((double)k + 0.5, m.dz));
    const double dx = __dadd_rn(cx, -s.pos[0]), dy = __dadd_rn(cy, -s.pos[1]), dz = __dadd_rn(cz, -s.pos[2]);
    bool inside = in_mesh;
    if (!s.isotropic) {
        const double a = __dadd_rn(__dadd_rn(__dmul_rn(dx, s.axis[0]), __dmul_rn(dy, s.axis[1])), __dmul_rn(dz, s.axis[2]));
        const double u = __dadd_rn(__dadd_rn(__dmul_rn(dx, s.up[0]), __dmul_rn(dy, s.up[1])), __dmul_rn(dz, s.up[2]));
        const double v = __dadd_rn(__dadd_rn(__dmul_rn(dx, s.side[0]), __dmul_rn(dy, s.side[1])), __dmul_rn(dz, s.side[2]));
        inside = in_mesh && a > 0.0 && fabs(u) <= __dmul_rn(a, s.tan_cone) && fabs(v) <= __dmul_rn(a, s.tan_fan);
    }
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double r = sqrt(r2);
    for (int t = 0; t < n_mat; ++t) s_len[t][threadIdx.x] = 0.0;
    if (inside) {

    // Walk from the centre (beta = 0) towards the source (beta = 1): direction e = s - c = -d. Everything per axis
    // lives in scalars and the axis of the next crossing is applied with selects: dynamically indexed arrays would
    // sit in local memory (the first version: 160 bytes of stack, several local loads and stores per step).
    // The next-crossing parameters advance by a constant per axis (fp64: <= 1e-13 after a few hundred steps).
    const double ex = -dx, ey = -dy, ez = -dz;
    const int sx = ex > 0.0 ? 1 : -1, sy = ey > 0.0 ? 1 : -1, sz = ez > 0.0 ? 1 : -1;
    double bx = 1e300, by = 1e300, bz = 1e300, dbx = 0.0, dby = 0.0, dbz = 0.0;
    if (ex != 0.0) { const double inv = 1.0 / ex; bx = (m.x0 + (i + (sx > 0 ? 1 : 0)) * m.dx - cx) * inv; dbx = fabs(m.dx * inv); }
    if (ey != 0.0) { const double inv = 1.0 / ey; by = (m.y0 + (j + (sy > 0 ? 1 : 0)) * m.dy - cy) * inv; dby = fabs(m.dy * inv); }
    if (ez != 0.0) { const double inv = 1.0 / ez; bz = (m.z0 + (k + (sz > 0 ? 1 : 0)) * m.dz - cz) * inv; dbz = fabs(m.dz * inv); }
    int ix = i, iy = j, iz = k;
    const long long px = sx, py = (long long)sy * m.nx, pz = (long long)sz * m.nx * m.ny;
    int cur = mat[cell];
    if (cur >= n_mat) { atomicExch(errflag, 1); cur = 0; }
    double run0 = 0.0;
    long long pos = (long long)cell;
    for (;;) {
        const bool ax = bx <= by && bx <= bz, ay = !ax && by <= bz;          // ties: x, then y, then z
        const double b = ax ? bx : (ay ? by : bz);
        if (b >= 1.0) { s_len[cur][threadIdx.x] += (1.0 - run0) * r; break; }      // source inside this cell
        if (ax) { ix += sx; bx += dbx; pos += px; }
        else if (ay) { iy += sy; by += dby; pos += py; }
        else { iz += sz; bz += dbz; pos += pz; }
        if ((unsigned)ix >= (unsigned)m.nx || (unsigned)iy >= (unsigned)m.ny || (unsigned)iz >= (unsigned)m.nz) {
            s_len[cur][threadIdx.x] += (b - run0) * r;                              // left the mesh
            break;
        }
        int nm = mat[pos];
        if (nm >= n_mat) { atomicExch(errflag, 1); nm = 0; }
        if (nm != cur) {
            s_len[cur][threadIdx.x] += (b - run0) * r;
            run0 = b;
            cur = nm;
        }
    }
    }
    __syncwarp();
    const double geo = 1.0 / (4.0 * 3.14159265358979323846 * r2);
    for (int g = 0; g < G; ++g) {
        double tau = 0.0;
        for (int t = 0; t < n_mat; ++t) tau += (double)sig_t_gm[g * n_mat + t] * s_len[t][threadIdx.x];
        const float v = inside ? (float)(spectrum.s[g] * exp(-tau) * geo) : 0.f;      // outside the beam: exactly 0 (R16)
        if (in_mesh) phi_u[(size_t)g * nv + cell] = v;
    }
}

// Y_lm of a direction, trig-free (same formulation as host_ylm in dos_api.cu), fp64 -> fp32.
template <int L>
__device__ __forceinline__ void dev_ylm(double mu, double eta, double xi, float *y)
{
    double re = 1.0, im = 0.0, dfact = 1.0;
#pragma unroll
    for (int mm = 0; mm <= L; ++mm) {
        if (mm > 0) {
            const double nre = re * mu - im * eta, nim = re * eta + im * mu;
            re = nre; im = nim;
            dfact *= (2.0 * mm - 1.0);
        }
        double t2 = 0.0, t1 = 0.0;
#pragma unroll
        for (int l = mm; l <= L; ++l) {
            double t;
            if (l == mm) t = dfact;
            else if (l == mm + 1) t = (2.0 * mm + 1.0) * xi * t1;
            else t = ((2.0 * l - 1.0) * xi * t1 - (l + mm - 1.0) * t2) / (double)(l - mm);
            t2 = t1; t1 = t;
            if (mm == 0) { y[l * (l + 1)] = (float)t; continue; }
            double f = 2.0;
            for (int q = l - mm + 1; q <= l + mm; ++q) f /= (double)q;
            const double nrm = sqrt(f);
            y[l * (l + 1) + mm] = (float)(nrm * t * re);
            y[l * (l + 1) - mm] = (float)(nrm * t * im);
        }
    }
}

}  // namespace

cudaError_t dos_launch_raytrace(const MeshDev &m, const SourceDev &s, const uint8_t *mat, int n_mat, int G,
                                const float *sig_t_gm, const SpectrumDev &spectrum, float *phi_u, int *errflag,
                                cudaStream_t st)
{
    const size_t nv = (size_t)m.nx * m.ny * m.nz;
    const unsigned grid = (unsigned)((nv + RT_THREADS - 1) / RT_THREADS);
    raytrace_kernel<<<grid, RT_THREADS, 0, st>>>(m, s, mat, n_mat, G, sig_t_gm, spectrum, phi_u, errflag);
    return cudaGetLastError();
}

namespace {

// ------------------------------------------------------------------------------------------------
// a2 + a3. Fixed source of group g (PAPER.md:49 first-collision source; eq. 2 g' sum):
//   Q_fix[lm] = Y_lm(Omega_r) sum_{g'<=g} sig_sl^{g'->g} phi_u^{g'} + sum_{g_lo<=g'<g} sig_sl^{g'->g} phi^{g'}[lm]
// One thread per cell; the cell's moments are MP/4 float4s. sig_s [n_mat][n_leg+1][G][G].
// ------------------------------------------------------------------------------------------------
template <int L>
__global__ void __launch_bounds__(128) group_source_kernel(MeshDev m, SourceDev s, const uint8_t *__restrict__ mat,
                                                           int n_mat, int G, int n_leg, int g, int g_lo,
                                                           const float *__restrict__ sig_s,
                                                           const float *__restrict__ phi_u,
                                                           const float *__restrict__ um,
                                                           const float *__restrict__ phi_all, float *__restrict__ qfix)
{
    constexpr int M = (L + 1) * (L + 1), MP = (M + 3) & ~3;
    const size_t nv = (size_t)m.nx * m.ny * m.nz;
    const size_t cell = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= nv) return;
    const int mt = min((int)mat[cell], n_mat - 1);       // ids are validated once per grid (validate_material_kernel); never index past a table
    const float *ss = sig_s + (size_t)mt * (n_leg + 1) * G * G;     // [l][from][to]
    float acc[MP];
#pragma unroll
    for (int t = 0; t < MP; ++t) acc[t] = 0.f;
    // first-collision part: s_l = sum_{g'<=g} sig_sl^{g'->g} phi_u^{g'}
    float sl[L + 1];
    bool any = false;
#pragma unroll
    for (int l = 0; l <= L; ++l) sl[l] = 0.f;
    for (int gp = 0; um == nullptr && gp <= g; ++gp) {
        const float pu = phi_u[(size_t)gp * nv + cell];
        if (pu != 0.f) {
            any = true;
#pragma unroll
            for (int l = 0; l <= L; ++l) sl[l] = fmaf(ss[((size_t)l * G + gp) * G + g], pu, sl[l]);
        }
    }
    if (any) {
        const int i = (int)(cell % m.nx), j = (int)((cell / m.nx) % m.ny), k = (int)(cell / ((size_t)m.nx * m.ny));
        const double dx = m.x0 + (i + 0.5) * m.dx - s.pos[0], dy = m.y0 + (j + 0.5) * m.dy - s.pos[1],
                     dz = m.z0 + (k + 0.5) * m.dz - s.pos[2];
        const double rinv = rsqrt(dx * dx + dy * dy + dz * dz);
        float y[M];
        dev_ylm<L>(dx * rinv, dy * rinv, dz * rinv, y);
#pragma unroll
        for (int l = 0; l <= L; ++l)
#pragma unroll
            for (int mm = -l; mm <= l; ++mm) acc[l * (l + 1) + mm] = y[l * (l + 1) + mm] * sl[l];
    }
    // downscatter from the collided fluence of the groups above (banded); in summed-source mode
    // also the first-collision source from the uncollided moments U^{g'}[lm] = sum_p Y_lm(Omega_p) phi_u,p^{g'} of
    // all source positions, g' <= g
    for (int pass = (um ? 0 : 1); pass < 2; ++pass)
    for (int gp = g_lo; gp < g + (pass == 0 ? 1 : 0); ++gp) {
        const float4 *pp = reinterpret_cast<const float4 *>((pass == 0 ? um : phi_all) + ((size_t)gp * nv + cell) * MP);
        float sg[L + 1];
#pragma unroll
        for (int l = 0; l <= L; ++l) sg[l] = ss[((size_t)l * G + gp) * G + g];
#pragma unroll
        for (int v = 0; v < MP / 4; ++v) {
            const float4 p4 = pp[v];
            const float pv[4] = {p4.x, p4.y, p4.z, p4.w};
#pragma unroll
            for (int t = 0; t < 4; ++t) {
                const int lm = 4 * v + t;
                if (lm < M) {
                    const int l = lm < 1 ? 0 : lm < 4 ? 1 : lm < 9 ? 2 : lm < 16 ? 3 : lm < 25 ? 4 : 5;
                    acc[lm] = fmaf(sg[l], pv[t], acc[lm]);
                }
            }
        }
    }
    float4 *qp = reinterpret_cast<float4 *>(qfix + cell * MP);
#pragma unroll
    for (int v = 0; v < MP / 4; ++v) qp[v] = make_float4(acc[4 * v], acc[4 * v + 1], acc[4 * v + 2], acc[4 * v + 3]);
}

// ------------------------------------------------------------------------------------------------
// a4. In-group source of one iteration: Q = Q_fix + sig_sl^{g->g} phi^(it-1); phi = 0 (the sweep then
// accumulates phi^(it) into it). One thread per float4 of a cell's moments. Also resets the sweep's
// hand-off flags and work-queue head.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) source_update_kernel(size_t nv, int MV, int M, const uint8_t *__restrict__ mat,
                                                            int n_mat, int G, int n_leg, int g, const float *__restrict__ sig_s,
                                                            const float4 *__restrict__ qfix, float4 *__restrict__ phi,
                                                            float4 *__restrict__ q, int first, int *done, int n_flags,
                                                            int *queue, float *__restrict__ phi00_old, size_t slot_stride)
{
    // blockIdx.y = problem of the position batch: its buffers sit slot_stride bytes x blockIdx.y further on
    {
        const size_t sh = (size_t)blockIdx.y * slot_stride;
        qfix = reinterpret_cast<const float4 *>(reinterpret_cast<const char *>(qfix) + sh);
        phi = reinterpret_cast<float4 *>(reinterpret_cast<char *>(phi) + sh);
        q = reinterpret_cast<float4 *>(reinterpret_cast<char *>(q) + sh);
        done = reinterpret_cast<int *>(reinterpret_cast<char *>(done) + sh);
        if (phi00_old) phi00_old = reinterpret_cast<float *>(reinterpret_cast<char *>(phi00_old) + sh);
    }
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < (size_t)n_flags) done[t] = 0;
    if (t == 0 && blockIdx.y == 0) *queue = 0;
    if (t >= nv * MV) return;
    const size_t cell = t / MV;
    const int v = (int)(t - cell * MV);
    float4 out = qfix[t];
    if (phi00_old && v == 0) phi00_old[cell] = first ? 0.f : phi[t].x;      // scalar fluence of the previous iterate (dos_solve_tol)
    if (!first) {
        const float *ss = sig_s + (size_t)min((int)mat[cell], n_mat - 1) * (n_leg + 1) * G * G + (size_t)g * G + g;   // + l*G*G
        const float4 p = phi[t];
        const float pv[4] = {p.x, p.y, p.z, p.w};
        float ov[4] = {out.x, out.y, out.z, out.w};
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int lm = 4 * v + e;
            if (lm < M) {
                const int l = lm < 1 ? 0 : lm < 4 ? 1 : lm < 9 ? 2 : lm < 16 ? 3 : lm < 25 ? 4 : 5;
                ov[e] = fmaf(ss[(size_t)l * G * G], pv[e], ov[e]);
            }
        }
        out = make_float4(ov[0], ov[1], ov[2], ov[3]);
    }
    q[t] = out;
    phi[t] = make_float4(0.f, 0.f, 0.f, 0.f);
}

// a8. phi_c^g = phi^g[00]; phi^g = phi_u^g + phi_c^g
__global__ void fluence_kernel(size_t nv, int G, int MP, const float *__restrict__ phi_u,
                               const float *__restrict__ phi_all, float *phi_c_out, float *phi_tot_out)
{
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nv * G) return;
    const float pc = phi_all[t * MP];
    if (phi_c_out) phi_c_out[t] = pc;
    if (phi_tot_out) phi_tot_out[t] = phi_u[t] + pc;
}

// a8. D(c) = sum_g K[m(c)][g] (phi_u^g + phi_c^g)(c); groups summed in index order
__global__ void dose_kernel(size_t nv, const uint8_t *__restrict__ mat, int n_mat, int G, int MP, const float *__restrict__ kerma,
                            const float *__restrict__ phi_u, const float *__restrict__ phi_all, float *dose,
                            int accumulate)
{
    const size_t cell = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= nv) return;
    const float *kr = kerma + (size_t)min((int)mat[cell], n_mat - 1) * G;
    float d = 0.f;
    for (int g = 0; g < G; ++g) d = fmaf(kr[g], phi_u[(size_t)g * nv + cell] + phi_all[((size_t)g * nv + cell) * MP], d);
    dose[cell] = accumulate ? dose[cell] + d : d;
}

}  // namespace

cudaError_t dos_launch_group_source(const MeshDev &m, const SourceDev &s, const uint8_t *mat, int n_mat, int G, int n_leg, int L,
                                    int g, int g_lo, const float *sig_s, const float *phi_u, const float *um,
                                    const float *phi_all, float *qfix, cudaStream_t st)
{
    const size_t nv = (size_t)m.nx * m.ny * m.nz;
    const unsigned grid = (unsigned)((nv + 127) / 128);
    switch (L) {
        case 0: group_source_kernel<0><<<grid, 128, 0, st>>>(m, s, mat, n_mat, G, n_leg, g, g_lo, sig_s, phi_u, um, phi_all, qfix); break;
        case 1: group_source_kernel<1><<<grid, 128, 0, st>>>(m, s, mat, n_mat, G, n_leg, g, g_lo, sig_s, phi_u, um, phi_all, qfix); break;
        case 2: group_source_kernel<2><<<grid, 128, 0, st>>>(m, s, mat, n_mat, G, n_leg, g, g_lo, sig_s, phi_u, um, phi_all, qfix); break;
        case 3: group_source_kernel<3><<<grid, 128, 0, st>>>(m, s, mat, n_mat, G, n_leg, g, g_lo, sig_s, phi_u, um, phi_all, qfix); break;
        case 4: group_source_kernel<4><<<grid, 128, 0, st>>>(m, s, mat, n_mat, G, n_leg, g, g_lo, sig_s, phi_u, um, phi_all, qfix); break;
        case 5: group_source_kernel<5><<<grid, 128, 0, st>>>(m, s, mat, n_mat, G, n_leg, g, g_lo, sig_s, phi_u, um, phi_all, qfix); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t dos_launch_source_update(size_t nv, const uint8_t *mat, int n_mat, int G, int n_leg, int L, int g, const float *sig_s,
                                     const float *qfix, float *phi, float *q, int first, int *done, int n_flags,
                                     int *queue, float *phi00_old, int n_batch, size_t slot_stride, cudaStream_t st)
{
    const int M = (L + 1) * (L + 1), MV = dos_mpad(L) / 4;
    size_t n = nv * MV;
    if ((size_t)n_flags > n) n = (size_t)n_flags;
    const unsigned grid = (unsigned)((n + 255) / 256);
    source_update_kernel<<<dim3(grid, (unsigned)n_batch), 256, 0, st>>>(nv, MV, M, mat, n_mat, G, n_leg, g, sig_s, (const float4 *)qfix,
                                                                        (float4 *)phi, (float4 *)q, first, done, n_flags, queue, phi00_old,
                                                                        slot_stride);
    return cudaGetLastError();
}

// Stopping measure of dos_solve_tol: out[0] = max_c |phi00_new - phi00_old|, out[1] = max_c |phi00_new| (as the bit
// patterns of non-negative floats, which order like integers; out must be zeroed before the launch).
namespace {
__global__ void __launch_bounds__(256) conv_kernel(size_t nv, int MP, const float *__restrict__ phi, const float *__restrict__ phi00_old, int *out)
{
    float d = 0.f, a = 0.f;
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < nv; c += (size_t)gridDim.x * blockDim.x) {
        const float v = phi[c * MP];
        d = fmaxf(d, fabsf(v - phi00_old[c]));
        a = fmaxf(a, fabsf(v));
    }
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
        d = fmaxf(d, __shfl_xor_sync(0xffffffffu, d, s));
        a = fmaxf(a, __shfl_xor_sync(0xffffffffu, a, s));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMax(out, __float_as_int(d));
        atomicMax(out + 1, __float_as_int(a));
    }
}
}  // namespace

cudaError_t dos_launch_conv(size_t nv, int MP, const float *phi, const float *phi00_old, int *out2, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(out2, 0, 2 * sizeof(int), st);
    if (e != cudaSuccess) return e;
    const unsigned grid = (unsigned)((nv + 255) / 256 < 1184 ? (nv + 255) / 256 : 1184);
    conv_kernel<<<grid, 256, 0, st>>>(nv, MP, phi, phi00_old, out2);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Summed-source mode (the cone beams of a CT scan form ONE source and are swept
// once). After the ray trace of position p: U^g[lm](c) (+)= Y_lm(Omega_p(c)) phi_u,p^g(c) and
// phi_u_sum^g(c) (+)= phi_u,p^g(c). One thread per cell; `first` overwrites instead of adding.
// ------------------------------------------------------------------------------------------------
template <int L>
__global__ void __launch_bounds__(128) um_accumulate_kernel(MeshDev m, SourceDev s, int G, int first,
                                                            const float *__restrict__ phi_u_pos, float *__restrict__ um,
                                                            float *__restrict__ phi_u_sum)
{
    constexpr int M = (L + 1) * (L + 1), MP = (M + 3) & ~3;
    const size_t nv = (size_t)m.nx * m.ny * m.nz;
    const size_t cell = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= nv) return;
    bool any = false;
    for (int g = 0; g < G; ++g) any |= phi_u_pos[(size_t)g * nv + cell] != 0.f;
    if (!any && !first) return;
    float y[MP];
#pragma unroll
    for (int t = 0; t < MP; ++t) y[t] = 0.f;
    if (any) {
        const int i = (int)(cell % m.nx), j = (int)((cell / m.nx) % m.ny), k = (int)(cell / ((size_t)m.nx * m.ny));
        const double dx = m.x0 + (i + 0.5) * m.dx - s.pos[0], dy = m.y0 + (j + 0.5) * m.dy - s.pos[1],
                     dz = m.z0 + (k + 0.5) * m.dz - s.pos[2];
        const double rinv = rsqrt(dx * dx + dy * dy + dz * dz);
        float yy[M];
        dev_ylm<L>(dx * rinv, dy * rinv, dz * rinv, yy);
#pragma unroll
        for (int t = 0; t < M; ++t) y[t] = yy[t];
    }
    for (int g = 0; g < G; ++g) {
        const float pu = phi_u_pos[(size_t)g * nv + cell];
        float4 *up = reinterpret_cast<float4 *>(um + ((size_t)g * nv + cell) * MP);
        float *ps = phi_u_sum + (size_t)g * nv + cell;
        if (first) {
            *ps = pu;
#pragma unroll
            for (int v = 0; v < MP / 4; ++v) up[v] = make_float4(y[4 * v] * pu, y[4 * v + 1] * pu, y[4 * v + 2] * pu, y[4 * v + 3] * pu);
        } else if (pu != 0.f) {
            *ps += pu;
#pragma unroll
            for (int v = 0; v < MP / 4; ++v) {
                float4 u = up[v];
                u.x = fmaf(y[4 * v], pu, u.x); u.y = fmaf(y[4 * v + 1], pu, u.y);
                u.z = fmaf(y[4 * v + 2], pu, u.z); u.w = fmaf(y[4 * v + 3], pu, u.w);
                up[v] = u;
            }
        }
    }
}

cudaError_t dos_launch_um_accumulate(const MeshDev &m, const SourceDev &s, int G, int L, int first, const float *phi_u_pos,
                                     float *um, float *phi_u_sum, cudaStream_t st)
{
    const size_t nv = (size_t)m.nx * m.ny * m.nz;
    const unsigned grid = (unsigned)((nv + 127) / 128);
    switch (L) {
        case 0: um_accumulate_kernel<0><<<grid, 128, 0, st>>>(m, s, G, first, phi_u_pos, um, phi_u_sum); break;
        case 1: um_accumulate_kernel<1><<<grid, 128, 0, st>>>(m, s, G, first, phi_u_pos, um, phi_u_sum); break;
        case 2: um_accumulate_kernel<2><<<grid, 128, 0, st>>>(m, s, G, first, phi_u_pos, um, phi_u_sum); break;
        case 3: um_accumulate_kernel<3><<<grid, 128, 0, st>>>(m, s, G, first, phi_u_pos, um, phi_u_sum); break;
        case 4: um_accumulate_kernel<4><<<grid, 128, 0, st>>>(m, s, G, first, phi_u_pos, um, phi_u_sum); break;
        case 5: um_accumulate_kernel<5><<<grid, 128, 0, st>>>(m, s, G, first, phi_u_pos, um, phi_u_sum); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

// Whole-grid check of the material ids (dos.h: "values < n_mat"), run once per grid: errflag[0] = 1 if any id >= n_mat.
namespace {
__global__ void validate_material_kernel(size_t nv, const uint8_t *__restrict__ mat, int n_mat, int *errflag)
{
    const size_t i = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) * 16;
    if (i >= nv) return;
    bool bad = false;
    if (i + 16 <= nv && (((uintptr_t)(mat + i)) & 15) == 0) {
        const uint4 v = *reinterpret_cast<const uint4 *>(mat + i);
        const unsigned w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int e = 0; e < 4; ++e)
#pragma unroll
            for (int b = 0; b < 4; ++b) bad |= (int)((w[e] >> (8 * b)) & 0xffu) >= n_mat;
    } else {
        for (size_t t = i; t < nv && t < i + 16; ++t) bad |= (int)mat[t] >= n_mat;
    }
    if (bad) atomicExch(errflag, 1);
}
}  // namespace

cudaError_t dos_launch_validate_material(size_t nv, const uint8_t *mat, int n_mat, int *errflag, cudaStream_t st)
{
    const size_t n = (nv + 15) / 16;
    validate_material_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(nv, mat, n_mat, errflag);
    return cudaGetLastError();
}

cudaError_t dos_launch_fluence(size_t nv, int G, int MP, const float *phi_u, const float *phi_all, float *phi_c_out,
                               float *phi_tot_out, cudaStream_t st)
{
    const unsigned grid = (unsigned)((nv * G + 255) / 256);
    fluence_kernel<<<grid, 256, 0, st>>>(nv, G, MP, phi_u, phi_all, phi_c_out, phi_tot_out);
    return cudaGetLastError();
}

cudaError_t dos_launch_dose(size_t nv, const uint8_t *mat, int n_mat, int G, int MP, const float *kerma,
                            const float *phi_u, const float *phi_all, float *dose, int accumulate, cudaStream_t st)
{
    const unsigned grid = (unsigned)((nv + 255) / 256);
    dose_kernel<<<grid, 256, 0, st>>>(nv, mat, n_mat, G, MP, kerma, phi_u, phi_all, dose, accumulate);
    return cudaGetLastError();
}
