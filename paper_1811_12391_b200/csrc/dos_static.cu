// dos_static.cu -- dos_uncollided_static: the uncollided ray trace (a1) for callers that cannot
// allocate device memory and therefore cannot hand the library a workspace (code under CUDA graph capture, tight
// serving loops, harnesses that forbid cudaMalloc). The ray-trace kernel's scratch -- its [G][n_mat] table of total
// cross sections and its bad-material flag, which every other entry point keeps in the caller's workspace -- lives in
// a file-scope __device__ array of DOS_STATIC_SCRATCH_BYTES instead. Every GPU that loads libdos.so holds that array
// until the process exits. The kernel is the one dos_uncollided launches (dos_kernels.cu), unchanged.
//
// The array is SHARED by every call and keeps the last call's contents: each call rewrites the part of the table it
// uses and clears the flag, on the caller's stream, before the kernel. Calls that overlap on the GPU (different streams
// without an ordering between them, several host threads) race on it; calls on one stream are safe.
// No cudaMalloc, cudaFree or allocating library routine is called here.
#include <cmath>
#include <mutex>
#include <string>

#include "../../include/dos.h"
#include "dos_internal.h"
#include "dos_kernels.h"

// scratch layout: [0, TABLE) float sig_t_gm[G][n_mat] | [TABLE, TABLE + 256) int flags[4] (flags[0]: material id >= n_mat met)
#define DOS_STATIC_TABLE_BYTES (DOS_MAX_G * DOS_MAX_MAT * 4)
static_assert(DOS_STATIC_SCRATCH_BYTES == DOS_STATIC_TABLE_BYTES + 256, "include/dos.h states the scratch size");

static __device__ __align__(256) unsigned char g_static_scratch[DOS_STATIC_SCRATCH_BYTES];

namespace {

struct SigTab {                       // host table, transposed to the kernel's [G][n_mat] order; travels by value
    float v[DOS_MAX_G * DOS_MAX_MAT];
};

// Device code of this file names the array directly (host code must not: there the name is a host-side stand-in).
__global__ void static_fill_kernel(SigTab tab, int n)
{
    float *t = reinterpret_cast<float *>(g_static_scratch);
    for (int i = threadIdx.x; i < n; i += blockDim.x) t[i] = tab.v[i];
    int *flags = reinterpret_cast<int *>(g_static_scratch + DOS_STATIC_TABLE_BYTES);
    if (threadIdx.x < 4) flags[threadIdx.x] = 0;          // the kernel only ever SETS the flag
}

// the array's device address, looked up once per device with that device current
constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
unsigned char *g_ptr[MAX_DEVICES];
bool g_have[MAX_DEVICES];
thread_local std::string g_static_err;

cudaError_t scratch_of_current_device(unsigned char **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_have[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_ptr[dev] = static_cast<unsigned char *>(p);
        g_have[dev] = true;
    }
    *out = g_ptr[dev];
    return cudaSuccess;
}

dos_status sfail(dos_status s, const std::string &msg)
{
    g_static_err = msg;
    return s;
}

}  // namespace

extern "C" const char *dos_static_last_error(void) { return g_static_err.c_str(); }

extern "C" dos_status dos_uncollided_static(const dos_mesh *mesh, const uint8_t *d_material_ids, int32_t n_mat, int32_t n_group,
                                            const float *sigma_t, const dos_source *source, const float *spectrum,
                                            float *d_phi_u_out, int32_t *d_bad_material_out, void *cuda_stream)
{
    if (!mesh || !d_material_ids || !sigma_t || !source || !spectrum || !d_phi_u_out) return sfail(DOS_ERR_INVALID_ARG, "null argument");
    if (mesh->nx < 1 || mesh->ny < 1 || mesh->nz < 1) return sfail(DOS_ERR_SHAPE, "mesh dimensions must be >= 1");
    if (!(mesh->dx > 0.0) || !(mesh->dy > 0.0) || !(mesh->dz > 0.0)) return sfail(DOS_ERR_INVALID_ARG, "voxel spacing must be > 0");
    // the limit of this entry point: the table must fit the static scratch
    if (n_mat < 1 || n_group < 1 || n_mat > DOS_MAX_MAT || n_group > DOS_MAX_G ||
        (size_t)n_mat * (size_t)n_group * sizeof(float) > (size_t)DOS_STATIC_TABLE_BYTES)
        return sfail(DOS_ERR_UNSUPPORTED, "dos_uncollided_static: n_mat x n_group = " + std::to_string(n_mat) + " x " + std::to_string(n_group) +
                                              " exceeds the static scratch (at most " + std::to_string(DOS_MAX_MAT) + " materials x " +
                                              std::to_string(DOS_MAX_G) + " groups, " + std::to_string(DOS_STATIC_SCRATCH_BYTES) + " bytes)");
    SigTab tab;
    for (int m = 0; m < n_mat; ++m)
        for (int g = 0; g < n_group; ++g) {
            const float s = sigma_t[(size_t)m * n_group + g];
            if (!(s > 0.f)) return sfail(DOS_ERR_INVALID_ARG, "sigma_t must be > 0");
            tab.v[(size_t)g * n_mat + m] = s;
        }
    auto dot = [](const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; };
    if (!source->isotropic) {
        if (std::fabs(dot(source->axis, source->axis) - 1.0) > 1e-9 || std::fabs(dot(source->up, source->up) - 1.0) > 1e-9 ||
            std::fabs(dot(source->axis, source->up)) > 1e-9)
            return sfail(DOS_ERR_INVALID_ARG, "axis and up must be orthonormal");
        if (!(source->tan_half_fan >= 0.0) || !(source->tan_half_cone >= 0.0))
            return sfail(DOS_ERR_INVALID_ARG, "collimation tangents must be >= 0");
    }
    {   // a source closer than 1e-9 cm to a voxel centre has no defined direction (as dos_uncollided)
        const dos_mesh &m = *mesh;
        const double fx = (source->pos[0] - m.x0) / m.dx - 0.5, fy = (source->pos[1] - m.y0) / m.dy - 0.5,
                     fz = (source->pos[2] - m.z0) / m.dz - 0.5;
        const double rx = std::nearbyint(fx), ry = std::nearbyint(fy), rz = std::nearbyint(fz);
        if (rx >= 0 && rx < m.nx && ry >= 0 && ry < m.ny && rz >= 0 && rz < m.nz) {
            const double ex = (fx - rx) * m.dx, ey = (fy - ry) * m.dy, ez = (fz - rz) * m.dz;
            if (std::sqrt(ex * ex + ey * ey + ez * ez) < 1e-9) return sfail(DOS_ERR_INVALID_ARG, "source coincides with a voxel centre");
        }
    }
    SpectrumDev sp;
    for (int g = 0; g < DOS_MAX_G; ++g) sp.s[g] = 0.0;
    for (int g = 0; g < n_group; ++g) {
        if (!(spectrum[g] >= 0.f)) return sfail(DOS_ERR_INVALID_ARG, "spectrum must be >= 0");
        sp.s[g] = (double)spectrum[g];
    }
    MeshDev md;
    md.nx = mesh->nx; md.ny = mesh->ny; md.nz = mesh->nz;
    md.dx = mesh->dx; md.dy = mesh->dy; md.dz = mesh->dz;
    md.x0 = mesh->x0; md.y0 = mesh->y0; md.z0 = mesh->z0;
    SourceDev sd;
    for (int i = 0; i < 3; ++i) { sd.pos[i] = source->pos[i]; sd.axis[i] = source->axis[i]; sd.up[i] = source->up[i]; }
    sd.side[0] = source->axis[1] * source->up[2] - source->axis[2] * source->up[1];
    sd.side[1] = source->axis[2] * source->up[0] - source->axis[0] * source->up[2];
    sd.side[2] = source->axis[0] * source->up[1] - source->axis[1] * source->up[0];
    sd.tan_fan = source->tan_half_fan; sd.tan_cone = source->tan_half_cone; sd.isotropic = source->isotropic;

    unsigned char *scratch = nullptr;
    cudaError_t e = scratch_of_current_device(&scratch);
    if (e != cudaSuccess) return sfail(DOS_ERR_CUDA, std::string("dos_uncollided_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    static_fill_kernel<<<1, 256, 0, st>>>(tab, n_mat * n_group);       // table and cleared flag, by kernel parameter: no host buffer to outlive the call
    if ((e = cudaGetLastError()) != cudaSuccess) return sfail(DOS_ERR_CUDA, std::string("dos_uncollided_static: ") + cudaGetErrorString(e));
    int *flags = reinterpret_cast<int *>(scratch + DOS_STATIC_TABLE_BYTES);
    e = dos_launch_raytrace(md, sd, d_material_ids, n_mat, n_group, reinterpret_cast<const float *>(scratch), sp, d_phi_u_out, flags, st);
    if (e != cudaSuccess) return sfail(DOS_ERR_CUDA, std::string("dos_uncollided_static: ") + cudaGetErrorString(e));
    if (d_bad_material_out) {
        e = cudaMemcpyAsync(d_bad_material_out, flags, sizeof(int), cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) return sfail(DOS_ERR_CUDA, std::string("dos_uncollided_static: ") + cudaGetErrorString(e));
    }
    return DOS_OK;
}
