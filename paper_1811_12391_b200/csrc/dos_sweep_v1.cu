// dos_sweep_v1.cu -- FIRST version of the S_N transport sweep, kept selectable (option sweep_impl=1) for A/B
// measurements against dos_sweep.cu. The S_N transport sweep (eq. 2-3) for one group and one source
// iteration: moment-to-discrete, diamond-difference cell update with set-to-zero fixup (north_star;
// DESIGN.md readings R3, R11, R12), discrete-to-moment, all 8 octants in one launch.
//
// Mapping:
//   work item   = (octant, tile of 8 x 4 (j,k) columns), whole x range; items are taken from a queue in
//                 an order in which every item's upwind neighbours come earlier (tile diagonal major)
//   CTA         = one item at a time; its warps split the octant's angles (AG angles per warp)
//   lane        = one (j,k) column of the tile; it marches along x with its x-face flux in a register.
//                 Lane (jj,kk) is jj+kk cells behind lane (0,0), so the y/z-face fluxes it needs were
//                 produced one step earlier by lanes (jj-1,kk) / (jj,kk-1): warp shuffles, no barrier.
//   tile faces  = y/z-face fluxes crossing a tile boundary go through an L2-resident buffer, published
//                 every `chunk` cells with a release flag that the downwind item's warp polls.
//   moments     = each lane reads its cell's Q[lm] (float4s, prefetched one step ahead) and adds its
//                 angles' w Y psi with one vector reduction (red.global.add.v4.f32) per 4 moments.
// The angular flux psi never leaves registers.
#include "dos_internal.h"

namespace {

__device__ __forceinline__ int ld_acquire(const int *p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void st_release(int *p, int v)
{
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

__device__ __forceinline__ void red_add_v4(float *p, float4 v)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z),
                 "f"(v.w)
                 : "memory");
}

// Diamond-difference cell update with set-to-zero fixup and rebalance. pin/pout: x, y, z faces.
__device__ __forceinline__ float dd_update(float q, float st, float cx, float cy, float cz, float cs, float ix,
                                           float iy, float iz, float &ox, float &oy, float &oz)
{
    float num = fmaf(cx, ix, fmaf(cy, iy, fmaf(cz, iz, q)));
    float pc = num / (st + cs);
    ox = 2.f * pc - ix;
    oy = 2.f * pc - iy;
    oz = 2.f * pc - iz;
    if (ox < 0.f || oy < 0.f || oz < 0.f) {
        bool fx = false, fy = false, fz = false;
        for (;;) {
            bool ax = !fx && ox < 0.f, ay = !fy && oy < 0.f, az = !fz && oz < 0.f;
            if (!(ax || ay || az)) break;
            fx |= ax; fy |= ay; fz |= az;
            num = q + (fx ? 0.5f * cx : cx) * ix + (fy ? 0.5f * cy : cy) * iy + (fz ? 0.5f * cz : cz) * iz;
            float den = st + (fx ? 0.f : cx) + (fy ? 0.f : cy) + (fz ? 0.f : cz);
            pc = num / den;
            ox = fx ? 0.f : 2.f * pc - ix;
            oy = fy ? 0.f : 2.f * pc - iy;
            oz = fz ? 0.f : 2.f * pc - iz;
        }
    }
    return pc;
}

template <int MP, int AG>
__global__ void __launch_bounds__(384) sweep_kernel(const SweepArgs p)
{
    constexpr int MV = MP / 4;
    extern __shared__ float4 smem4[];
    float *s_m2d = reinterpret_cast<float *>(smem4);      // [A][MP] for the current octant
    float *s_d2m = s_m2d + p.per_oct * MP;                 // [A][MP]
    float *s_cdd = s_d2m + p.per_oct * MP;                 // [A][4]
    float *s_sig = s_cdd + p.per_oct * 4;                  // [n_mat]
    __shared__ int s_item;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int jj = lane & (DOS_TJ - 1), kk = lane / DOS_TJ;
    const int skew = jj + kk;
    const int nx = p.nx, ny = p.ny, nz = p.nz, A = p.per_oct;
    const int a0 = warp * AG;

    for (int t = threadIdx.x; t < A * 4; t += blockDim.x) s_cdd[t] = p.cdd[t];
    for (int t = threadIdx.x; t < p.n_mat; t += blockDim.x) s_sig[t] = p.sig_t[t];
    int cur_oct = -1;

    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_item = atomicAdd(p.queue, 1);
        __syncthreads();
        const int item = s_item;
        if (item >= p.n_items) break;
        const int packed = p.items[item];
        const int o = packed & 7, tj = (packed >> 3) & 0x3FFF, tk = packed >> 17;
        if (o != cur_oct) {
            for (int t = threadIdx.x; t < A * MP; t += blockDim.x) {
                s_m2d[t] = p.m2d[(size_t)o * A * MP + t];
                s_d2m[t] = p.d2m[(size_t)o * A * MP + t];
            }
            cur_oct = o;
            __syncthreads();
        }

        // ---- per-lane geometry of this item (oriented indices: primes sweep upwards) ----
        const int jp = tj * DOS_TJ + jj, kp = tk * DOS_TK + kk;
        const bool valid = jp < ny && kp < nz;
        const int j = (o & 2) ? ny - 1 - jp : jp;
        const int k = (o & 4) ? nz - 1 - kp : kp;
        const int istep = (o & 1) ? -1 : 1;
        const size_t cell0 = ((size_t)k * ny + j) * nx + ((o & 1) ? nx - 1 : 0);
        const bool load_y = valid && jj == 0 && tj > 0;
        const bool load_z = valid && kk == 0 && tk > 0;
        const bool store_y = valid && jj == DOS_TJ - 1 && tj < p.ntj - 1;
        const bool store_z = valid && kk == DOS_TK - 1 && tk < p.ntk - 1;
        const size_t ystride = (size_t)p.ntj * nz * nx, zstride = (size_t)p.ntk * ny * nx;
        const float *fy_in = p.fy + (((size_t)(o * A + a0) * p.ntj + (tj - 1)) * nz + kp) * nx;
        float *fy_out = p.fy + (((size_t)(o * A + a0) * p.ntj + tj) * nz + kp) * nx;
        const float *fz_in = p.fz + (((size_t)(o * A + a0) * p.ntk + (tk - 1)) * ny + jp) * nx;
        float *fz_out = p.fz + (((size_t)(o * A + a0) * p.ntk + tk) * ny + jp) * nx;
        const int id = (o * p.ntk + tk) * p.ntj + tj;
        int *my_flag = p.done + (size_t)id * p.n_grp + warp;
        const int *up_y = p.done + (size_t)(id - 1) * p.n_grp + warp;
        const int *up_z = p.done + (size_t)(id - p.ntj) * p.n_grp + warp;
        const bool dep_y = tj > 0, dep_z = tk > 0;
        int avail = (dep_y || dep_z) ? 0 : nx;    // cells along x whose upwind tile faces are published

        float px[AG], oy[AG], oz[AG];
#pragma unroll
        for (int r = 0; r < AG; ++r) px[r] = oy[r] = oz[r] = 0.f;

        float4 qn[MV];
        float byn[AG], bzn[AG];
        int matn = 0;
#pragma unroll
        for (int v = 0; v < MV; ++v) qn[v] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int r = 0; r < AG; ++r) byn[r] = bzn[r] = 0.f;

        const int T = nx + DOS_SKEW;
        for (int t = -1; t < T; ++t) {
            // ---- rotate the prefetched operands of step t into place ----
            float4 qc[MV];
            float byc[AG], bzc[AG];
#pragma unroll
            for (int v = 0; v < MV; ++v) qc[v] = qn[v];
#pragma unroll
            for (int r = 0; r < AG; ++r) { byc[r] = byn[r]; bzc[r] = bzn[r]; }
            const int matc = matn;

            // ---- prefetch step t+1 (needs the upwind faces of cell t+1 of the lead lane) ----
            if (t + 1 < T) {
                const int need = min(t + 2, nx);
                int spins = 0;
                while (avail < need) {
                    int ya = dep_y ? ld_acquire(up_y) : nx;
                    int za = dep_z ? ld_acquire(up_z) : nx;
                    avail = min(ya, za);
                    if (avail < need) {
                        __nanosleep(40);
                        // watchdog: a hand-off that never arrives must not hang the GPU; the result is
                        // then invalid and dos_check / dos_dose_host report DOS_ERR_CUDA
                        if (++spins > DOS_SPIN_LIMIT) atomicExch(p.abort_flag, 1);
                        if ((spins & 255) == 0 && ld_acquire(p.abort_flag)) avail = nx;
                    }
                }
                const int ipn = t + 1 - skew;
                if (valid && ipn >= 0 && ipn < nx) {
                    const size_t cell = cell0 + (ptrdiff_t)istep * ipn;
                    const float4 *qp = reinterpret_cast<const float4 *>(p.Q) + cell * MV;
#pragma unroll
                    for (int v = 0; v < MV; ++v) qn[v] = __ldg(qp + v);
                    matn = __ldg(p.mat + cell);
                    if (load_y) {
#pragma unroll
                        for (int r = 0; r < AG; ++r) byn[r] = __ldcg(fy_in + r * ystride + ipn);
                    }
                    if (load_z) {
#pragma unroll
                        for (int r = 0; r < AG; ++r) bzn[r] = __ldcg(fz_in + r * zstride + ipn);
                    }
                }
            }
            if (t < 0) continue;

            // ---- step t: this lane's cell is ip = t - skew ----
            const int ip = t - skew;
            const bool act = valid && ip >= 0 && ip < nx;
            float yin[AG], zin[AG];
#pragma unroll
            for (int r = 0; r < AG; ++r) {
                yin[r] = __shfl_up_sync(0xffffffffu, oy[r], 1);
                zin[r] = __shfl_up_sync(0xffffffffu, oz[r], DOS_TJ);
                if (jj == 0) yin[r] = load_y ? byc[r] : 0.f;     // tile inflow or vacuum
                if (kk == 0) zin[r] = load_z ? bzc[r] : 0.f;
            }
            if (act) {
                const size_t cell = cell0 + (ptrdiff_t)istep * ip;
                const float st = s_sig[matc];
                float q[AG], pc[AG];
#pragma unroll
                for (int r = 0; r < AG; ++r) q[r] = 0.f;
#pragma unroll
                for (int v = 0; v < MV; ++v) {
#pragma unroll
                    for (int r = 0; r < AG; ++r) {
                        const float4 c = *reinterpret_cast<const float4 *>(s_m2d + (a0 + r) * MP + 4 * v);
                        q[r] = fmaf(c.x, qc[v].x, fmaf(c.y, qc[v].y, fmaf(c.z, qc[v].z, fmaf(c.w, qc[v].w, q[r]))));
                    }
                }
#pragma unroll
                for (int r = 0; r < AG; ++r) {
                    const float4 c = *reinterpret_cast<const float4 *>(s_cdd + (a0 + r) * 4);
                    const float ix = (ip == 0) ? 0.f : px[r];
                    float ox, oyr, ozr;
                    pc[r] = dd_update(q[r], st, c.x, c.y, c.z, c.w, ix, yin[r], zin[r], ox, oyr, ozr);
                    px[r] = ox; oy[r] = oyr; oz[r] = ozr;
                    if (store_y) __stcg(fy_out + r * ystride + ip, oyr);
                    if (store_z) __stcg(fz_out + r * zstride + ip, ozr);
                }
                float *php = p.phi + cell * MP;
#pragma unroll
                for (int v = 0; v < MV; ++v) {
                    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                    for (int r = 0; r < AG; ++r) {
                        const float4 d = *reinterpret_cast<const float4 *>(s_d2m + (a0 + r) * MP + 4 * v);
                        acc.x = fmaf(d.x, pc[r], acc.x);
                        acc.y = fmaf(d.y, pc[r], acc.y);
                        acc.z = fmaf(d.z, pc[r], acc.z);
                        acc.w = fmaf(d.w, pc[r], acc.w);
                    }
                    red_add_v4(php + 4 * v, acc);
                }
            }
            // ---- publish: the slowest lane (skew DOS_SKEW) has just finished cell t - DOS_SKEW ----
            const int fin = t - DOS_SKEW;
            if (fin >= 0 && (((fin + 1) % p.chunk) == 0 || fin == nx - 1)) {
                __syncwarp();
                if (lane == 0) {
                    __threadfence();
                    st_release(my_flag, fin + 1);
                }
            }
        }
    }
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side: choice of angles per warp, occupancy-sized persistent grid, template dispatch
// ------------------------------------------------------------------------------------------------
typedef void (*sweep_fn)(const SweepArgs);

template <int MP>
static sweep_fn pick_ag(int ag)
{
    switch (ag) {
        case 1: return sweep_kernel<MP, 1>;
        case 2: return sweep_kernel<MP, 2>;
        case 3: return sweep_kernel<MP, 3>;
        case 4: return sweep_kernel<MP, 4>;
    }
    return nullptr;
}

static sweep_fn pick(int L, int ag)
{
    switch (dos_mpad(L)) {
        case 4: return pick_ag<4>(ag);
        case 12: return pick_ag<12>(ag);
        case 16: return pick_ag<16>(ag);
        case 28: return pick_ag<28>(ag);
        case 36: return pick_ag<36>(ag);
    }
    return nullptr;
}

static size_t sweep_smem(int L, int per_oct, int n_mat)
{
    return sizeof(float) * ((size_t)2 * per_oct * dos_mpad(L) + 4 * per_oct + n_mat + 4);
}

// Angles per warp: the largest of 4, 3, 2, 1 that divides the octant's angle count and keeps the CTA
// within 12 warps (S2: 1x1, S4: 3 -> 1 warp, S6: 6 -> 3x2, S8: 10 -> 5x2, S12: 21 -> 7x3, S16: 36 -> 9x4).
int dos_sweep_v1_angles_per_warp(int per_oct, int L)
{
    (void)L;
    int best = 0;
    for (int ag = 4; ag >= 1; --ag)
        if (per_oct % ag == 0 && per_oct / ag <= 12) { best = ag; break; }
    return best;
}

cudaError_t dos_sweep_v1_grid(int L, int ag, int per_oct, int n_mat, int n_items, int *grid_out)
{
    sweep_fn f = pick(L, ag);
    if (!f) return cudaErrorInvalidValue;
    const size_t smem = sweep_smem(L, per_oct, n_mat);
    cudaError_t e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 0, per_sm = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    const int threads = (per_oct / ag) * 32;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, f, threads, smem)) != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    // Persistent CTAs: every resident CTA pulls items until the queue is empty. All CTAs of the grid
    // must be co-resident only for speed, not for progress: an item never waits on a later item.
    int g = sms * per_sm;
    *grid_out = g < n_items ? g : n_items;
    return cudaSuccess;
}

cudaError_t dos_launch_sweep_v1(const SweepArgs &a, int L, int ag, int grid, cudaStream_t s)
{
    sweep_fn f = pick(L, ag);
    if (!f) return cudaErrorInvalidValue;
    const size_t smem = sweep_smem(L, a.per_oct, a.n_mat);
    f<<<grid, a.n_grp * 32, smem, s>>>(a);
    return cudaGetLastError();
}
