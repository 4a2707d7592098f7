// dos_sweep_ffma.cu -- the sweep with both contractions on the FP32 pipe (FFMA): the fallback for quadratures the
// tensor-memory sweep (dos_sweep_umma.cu) has no shape for, and the A/B partner of it (option "sweep_contraction" = 1).
//
// The S_N transport sweep (eq. 2-3) for one group and one source
// iteration: moment-to-discrete (a5), diamond-difference cell update with set-to-zero fixup and
// rebalance (a6; north_star; readings R3, R11, R12), discrete-to-moment (a7), all 8 octants
// in one launch. DESIGN.md section 6 has the mapping and the measurements behind it.
//
//   work item   (octant, tile of 8 x 4 (j,k) columns), whole x range. Items sit in a queue in an order
//               in which an item's two upwind tiles come earlier (tile-diagonal major); persistent
//               CTAs pop them.
//   CTA         all A angles of the octant for one tile: NW = A / AG compute warps (AG angles each)
//               plus one service warp that only polls and publishes hand-off flags.
//   lane        one (j,k) column; it marches along x with its x-face flux in a register. Lane (jj,kk)
//               is jj+kk cells behind lane (0,0) (KBA wavefront inside the warp), so the y/z-face
//               fluxes it needs left lanes (jj-1,kk) / (jj,kk-1) one step earlier: warp shuffles.
//   step        one x-advance of the whole CTA, closed by one __syncthreads.
//   staging     the step's 32 source-moment vectors Q[cell][MP] and its tile-inflow face fluxes are
//               copied into a shared-memory ring by cp.async DOS_PREFETCH steps ahead (one 16-byte
//               copy per thread per step), so no warp waits on L2/HBM inside a step.
//   moments     every warp leaves psi_c in shared memory; after the barrier the cell's w Y psi is
//               summed over ALL angles of the octant by (cell, 4-moment) threads and added to
//               phi[cell][lm] with one red.global.add.v4.f32 per cell, octant and 4 moments (the first
//               version issued one per warp: A/AG times as many).
//   tile faces  fluxes crossing a tile boundary go through an L2-resident buffer indexed by the
//               wavefront diagonal (d = x + kk for y faces, x + jj for z faces), so what a downwind
//               step needs is one contiguous block; published every `chunk` steps with a release
//               store that the downwind CTA's service warp acquires.
// The angular flux psi never leaves registers / shared memory.
#include "dos_internal.h"

namespace {

constexpr int DQ = DOS_PREFETCH_Q;    // steps between issuing the copy of a step's source moments and using them
constexpr int RQ = DOS_RING_Q;        // ring slots of the staged moments (power of two > DQ)
constexpr int DF = DOS_PREFETCH_F;    // the same for the tile-inflow faces (shorter: it delays a downwind tile's start)
constexpr int RF = DOS_RING_F;
constexpr int BIG = 1 << 30;
constexpr int FINW = DOS_TK + DOS_TJ;   // inflow floats per angle and step: 4 y faces then 8 z faces

__device__ __forceinline__ int ld_relaxed(const int *p)
{
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }

// flag-in-data hand-off (Sweep2Args::ll): one 8-byte store per face value, 16-byte polls of two pairs
__device__ __forceinline__ void st_pair(float *p, float v, unsigned epoch)
{
    asm volatile("st.relaxed.gpu.global.v2.b32 [%0], {%1, %2};" ::"l"(p), "r"(__float_as_uint(v)), "r"(epoch) : "memory");
}
__device__ __forceinline__ uint4 ld_pairs(const float *p)
{
    uint4 v;
    asm volatile("ld.relaxed.gpu.global.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}

// CTA-scope release / acquire on a shared-memory word (service warp <-> compute warps)
// (by 32-bit shared address, converted once per kernel: a generic-to-shared conversion inside a loop costs a read of a
// special register, SR_CgaCtaId, every time)
__device__ __forceinline__ void st_release_cta(unsigned a, int v)
{
    asm volatile("st.release.cta.shared.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ int ld_acquire_cta(unsigned a)
{
    int v;
    asm volatile("ld.acquire.cta.shared.s32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}

// shared-memory accesses through explicit 32-bit shared addresses (keeps the address arithmetic of the
// step loop to one integer add per access)
__device__ __forceinline__ unsigned smem_addr(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ float lds_f32(unsigned a)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ int lds_s32(unsigned a)
{
    int v;
    asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ float4 lds_v4(unsigned a)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts_f32(unsigned a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ void sts_s32(unsigned a, int v) { asm volatile("st.shared.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void sts_v4(unsigned a, float4 v)
{
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

// barrier of the compute warps only (the service warp never joins it)
__device__ __forceinline__ void bar_compute(int n_threads) { asm volatile("bar.sync 1, %0;" ::"r"(n_threads) : "memory"); }

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

// 16-byte asynchronous global -> shared copy that bypasses L1 (tile faces are written by other SMs
// during this launch; an L1 line could be stale)
__device__ __forceinline__ void cp_async16(unsigned smem_a, const void *gmem)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_a), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

// shared-memory row length of one cell's moments: MP floats, padded so that MPS/4 is odd and the
// per-lane LDS.128 of a warp (lane stride MPS floats) are bank-conflict free
__host__ __device__ constexpr int mps_of(int MP) { return ((MP / 4) & 1) ? MP : MP + 4; }

// Slow path of the cell update: at least one extrapolated outflow was negative. Faces found negative
// are pinned to zero together, the balance is re-solved, and the pinned set only grows (R12).
// in/out: pc, ox, oy, oz of the unfixed solve -> of the fixed one.
__device__ __forceinline__ void dd_fixup(float &pc, float &ox, float &oy, float &oz, float q, float st, float cx, float cy,
                                         float cz, float ix, float iy, float iz)
{
    const float hx = cx * ix, hy = cy * iy, hz = cz * iz;
    bool fx = false, fy = false, fz = false;
#pragma unroll 1
    do {
        fx |= ox < 0.f; fy |= oy < 0.f; fz |= oz < 0.f;       // a pinned face's outflow is 0 and never tests negative
        const float num = q + (fx ? 0.5f * hx : hx) + (fy ? 0.5f * hy : hy) + (fz ? 0.5f * hz : hz);
        const float den = st + (fx ? 0.f : cx) + (fy ? 0.f : cy) + (fz ? 0.f : cz);
        pc = __fdividef(num, den);
        ox = fx ? 0.f : 2.f * pc - ix;
        oy = fy ? 0.f : 2.f * pc - iy;
        oz = fz ? 0.f : 2.f * pc - iz;
    } while (fminf(ox, fminf(oy, oz)) < 0.f);
}

// One cp.async of 16 bytes that a thread issues every step: at step t it fetches what step s = t + dist
// needs (if s lies inside the window [lo, hi]) from src0 + s * sstep (floats) into ring slot s & mask.
struct LoadOp {
    const float *src0;
    unsigned dst0;         // shared-memory byte address of ring slot 0
    int sstep, dslot, lo, hi, dist, mask;      // dslot: bytes between ring slots
    int e0, nval;          // face ops: lane index (kk or jj) of the op's first value, lanes of the upwind tile inside the mesh
};

struct ItemGeom {
    int o, tj, tk, id;
    bool has_y, has_z;
    const float *fy_in, *fz_in;
};

// Decode load `op` of the current item: ops [0, 32 MV) fetch 4 moments of lane c's cell, the next A
// fetch the 4 y-face inflows of angle a, the last 2A the 8 z-face inflows of angle a in two halves.
template <int MP, bool LL>
__device__ __forceinline__ LoadOp make_op(int op, const Sweep2Args &p, const ItemGeom &g, float *s_q, float *s_fin)
{
    constexpr int MV = MP / 4, MPS = mps_of(MP);
    const int A = p.per_oct, nx = p.nx;
    LoadOp d;
    d.lo = 1; d.hi = 0;                      // empty window
    d.e0 = 0; d.nval = 0;
    d.src0 = p.Q; d.dst0 = smem_addr(s_q); d.sstep = 0; d.dslot = 0; d.dist = DQ; d.mask = RQ - 1;
    if (op < 32 * MV) {
        const int c = op / MV, v = op - c * MV;
        const int jj = c & (DOS_TJ - 1), kk = c / DOS_TJ, skew = jj + kk;
        const int jp = g.tj * DOS_TJ + jj, kp = g.tk * DOS_TK + kk;
        if (jp < p.ny && kp < p.nz) {
            const int j = (g.o & 2) ? p.ny - 1 - jp : jp, k = (g.o & 4) ? p.nz - 1 - kp : kp;
            const int istep = (g.o & 1) ? -1 : 1;
            const long long cell0 = ((long long)k * p.ny + j) * nx + ((g.o & 1) ? nx - 1 : 0);
            d.sstep = istep * MP;
            d.src0 = p.Q + (cell0 - (long long)istep * skew) * MP + 4 * v;
            d.lo = skew; d.hi = skew + nx - 1;
        }
        d.dst0 = smem_addr(s_q + c * MPS + 4 * v);
        d.dslot = 32 * MPS * 4;
    } else if (op < 32 * MV + A) {
        const int a = op - 32 * MV;
        if (g.has_y) { d.lo = 0; d.hi = nx + DOS_TK - 2; }
        d.src0 = g.fy_in + a * DOS_TK;
        d.sstep = A * DOS_TK;
        if (LL) { d.src0 = p.fy + 2 * (d.src0 - p.fy); d.sstep *= 2; }      // (value, epoch) pairs
        d.e0 = 0; d.nval = min(DOS_TK, p.nz - g.tk * DOS_TK);
        d.dst0 = smem_addr(s_fin + a * FINW);
        d.dslot = A * FINW * 4; d.dist = DF; d.mask = RF - 1;
    } else {
        const int idx = op - 32 * MV - A, a = idx >> 1, h = idx & 1;
        if (g.has_z) { d.lo = 0; d.hi = nx + DOS_TJ - 2; }
        d.src0 = g.fz_in + a * DOS_TJ + 4 * h;
        d.sstep = A * DOS_TJ;
        if (LL) { d.src0 = p.fz + 2 * (d.src0 - p.fz); d.sstep *= 2; }
        d.e0 = 4 * h; d.nval = min(DOS_TJ, p.ny - g.tj * DOS_TJ);
        d.dst0 = smem_addr(s_fin + a * FINW + DOS_TK + 4 * h);
        d.dslot = A * FINW * 4; d.dist = DF; d.mask = RF - 1;
    }
    return d;
}

// Warp roles inside a CTA (one work item at a time):
//   compute warps  [0, NW)        AG angles each: M2D, diamond difference, face hand-off, psi_c to smem
//   aux warps      [NW, NW + NX)  staging copies of the source moments (cp.async), D2M reduction + red.global
//                                 of the previous step
//   feeder warp    NW + NX        staging copies of the tile-inflow faces, material ids, step count for the
//                                 service warp
//   service warp   NW + NX + 1    global hand-off flags (never joins the per-step barrier)
// TMAX = CTA size bound for the register budget. LL = flag-in-data hand-off of the tile faces (Sweep2Args::ll; small
// meshes): an instance of its own, so that the large-mesh kernels carry none of it.
template <int MP, int AG, int TMAX, int MINB, bool LL>
__global__ void __launch_bounds__(TMAX, MINB) sweep_kernel(const Sweep2Args p0)
{
    Sweep2Args p = p0;       // Q, phi, fy, fz, done are re-pointed at the item's problem of the batch
    constexpr int MV = MP / 4, MPS = mps_of(MP);
    extern __shared__ float4 smem4[];
    const int A = p.per_oct, NW = p.n_warps, NX = p.n_aux;
    const int NB = (NW + NX + 1) * 32;                      // threads in the per-step barrier (compute, aux, tick)
    float *s_q = reinterpret_cast<float *>(smem4);          // [RQ][32][MPS] staged source moments
    float *s_fin = s_q + RQ * 32 * MPS;                     // [RF][A][FINW] staged tile-inflow faces
    float *s_psi = s_fin + RF * A * FINW;                   // [2][A][32]    psi_c of the last two steps
    float *s_m2d = s_psi + 2 * A * 32;                      // [A][MP] for the current octant
    float *s_d2m = s_m2d + A * MP;                          // [A][MP]
    float *s_cdd = s_d2m + A * MP;                          // [A][4]
    float *s_rden = s_cdd + A * 4;                          // [n_mat][A]  1 / (sigma_t + cx + cy + cz)
    float *s_sig = s_rden + p.n_mat * A;                    // [n_mat]
    int *s_mat = reinterpret_cast<int *>(s_sig + ((p.n_mat + 3) & ~3));   // [4][32] material ids of 4 steps
    __shared__ int s_item;
    __shared__ int s_done;        // steps finished by the compute/aux warps (written by one aux thread)
    __shared__ int s_allowed;     // last step whose tile-inflow faces are published upwind (service warp)

    // The thread index is read ONCE, through a volatile asm: left to itself the compiler re-reads the special register
    // (S2R, ~20 cycles) and re-derives lane / jj / kk wherever a loop uses them instead of holding a register -- measured
    // with ncu at config 4 (64-register variant): 15 % of all executed instructions came from these two source lines.
    int tid;
    asm volatile("mov.u32 %0, %%tid.x;" : "=r"(tid));
    const int lane = tid & 31, warp = tid >> 5;
    const unsigned a_done = smem_addr(&s_done), a_allowed = smem_addr(&s_allowed);
    const bool tick = warp == NW + NX, service = warp == NW + NX + 1, aux = warp >= NW && warp < NW + NX;
    const int jj = lane & (DOS_TJ - 1), kk = lane / DOS_TJ;
    const int skew = jj + kk;
    const int nx = p.nx, ny = p.ny, nz = p.nz;
    const int T = nx + DOS_SKEW;
    const size_t fstride_y = (size_t)(nx + DOS_FACE_PAD) * A * DOS_TK, fstride_z = (size_t)(nx + DOS_FACE_PAD) * A * DOS_TJ;

    for (int t = tid; t < p.n_mat; t += blockDim.x) s_sig[t] = p.sig_t[t];
    int cur_oct = -1;

    for (;;) {
        __syncthreads();                              // previous item finished with the staging buffers
        if (tid == 0) s_item = atomicAdd(p.queue, 1);
        __syncthreads();
        if (s_item >= p.n_items) break;
        const int item = s_item / p.n_batch;
        {
            const size_t sh = (size_t)(s_item - item * p.n_batch) * p.slot_stride;
            p.Q = reinterpret_cast<const float *>(reinterpret_cast<const char *>(p0.Q) + sh);
            p.phi = reinterpret_cast<float *>(reinterpret_cast<char *>(p0.phi) + sh);
            p.fy = reinterpret_cast<float *>(reinterpret_cast<char *>(p0.fy) + sh);
            p.fz = reinterpret_cast<float *>(reinterpret_cast<char *>(p0.fz) + sh);
            p.done = reinterpret_cast<int *>(reinterpret_cast<char *>(p0.done) + sh);
        }
        const int tile_item = item / p.a_split, part = item - tile_item * p.a_split;
        const int packed = p.items[tile_item];
        ItemGeom g;
        g.o = packed & 7; g.tj = (packed >> 3) & 0x3FFF; g.tk = packed >> 17;
        g.id = ((g.o * p.ntk + g.tk) * p.ntj + g.tj) * p.a_split + part;
        g.has_y = g.tj > 0; g.has_z = g.tk > 0;
        g.fy_in = p.fy + (g.has_y ? (size_t)(g.id - p.a_split) * fstride_y : 0);
        g.fz_in = p.fz + (g.has_z ? (size_t)(g.id - p.ntj * p.a_split) * fstride_z : 0);
        const int o = g.o;
        if (o * 8 + part != cur_oct) {
            // tables of this CTA's angles: [o][part * A, (part + 1) * A)
            const size_t abase = (size_t)o * p.per_oct_full + (size_t)part * A;
            for (int t = tid; t < A * MP; t += blockDim.x) {
                s_m2d[t] = p.m2d[abase * MP + t];
                s_d2m[t] = p.d2m[abase * MP + t];
            }
            for (int t = tid; t < A * 4; t += blockDim.x) s_cdd[t] = p.cdd[part * A * 4 + t];
            for (int t = tid; t < p.n_mat * A; t += blockDim.x) {
                const int m = t / A, a = t - m * A;
                s_rden[t] = 1.f / (p.sig_t[m] + p.cdd[(part * A + a) * 4 + 3]);
            }
            cur_oct = o * 8 + part;
        }

        if (service) {
            // ------- service warp: publishes this item's progress, follows the upwind items' progress -------
            // It never joins the per-step barrier, so the latency of its global loads, fences and stores
            // stays off the other warps' critical path; the two sides talk through s_done / s_allowed.
            const int *up_y = p.done + (g.has_y ? g.id - p.a_split : g.id), *up_z = p.done + (g.has_z ? g.id - p.ntj * p.a_split : g.id);
            int *my_flag = p.done + g.id;
            int avail_y = g.has_y ? 0 : BIG, avail_z = g.has_z ? 0 : BIG;
            if (lane == 0) {
                s_done = 0;
                s_allowed = (g.has_y || g.has_z) ? -1 : BIG;
            }
            __syncthreads();                          // S2
            if (LL) continue;                         // flag-in-data hand-off: the faces carry their own validity
            int published = 0, spins = 0;
            for (;;) {
                const int dn = ld_acquire_cta(a_done);
                if (dn - published >= p.chunk || (dn == T && published < T)) {
                    if (lane == 0) st_release(my_flag, dn);       // steps < dn are complete
                    published = dn;
                }
                if (published == T) break;
                if (avail_y < T || avail_z < T) {
                    const int vy = avail_y < T ? ld_relaxed(up_y) : avail_y;
                    const int vz = avail_z < T ? ld_relaxed(up_z) : avail_z;
                    if (vy != avail_y || vz != avail_z) {
                        fence_acq_rel_gpu();          // relaxed load + fence = acquire of the upwind release
                        avail_y = vy; avail_z = vz;
                        const int al = min(avail_y >= T ? BIG : avail_y - DOS_TJ, avail_z >= T ? BIG : avail_z - DOS_TK);
                        if (lane == 0) st_release_cta(a_allowed, al);
                        spins = 0;
                    } else {
                        // watchdog: a hand-off that never arrives must not hang the GPU; the result is then
                        // invalid and dos_check / dos_dose_host report DOS_ERR_CUDA
                        if (++spins > DOS_SPIN_LIMIT) atomicExch(p.abort_flag, 1);
                        if ((spins & 255) == 0 && ld_relaxed(p.abort_flag)) {
                            avail_y = avail_z = BIG;
                            if (lane == 0) st_release_cta(a_allowed, BIG);
                        }
                        __nanosleep(DOS_POLL_NS);
                    }
                } else {
                    __nanosleep(2 * DOS_POLL_NS);
                }
            }
            continue;
        }

        // geometry of this lane's (j,k) column: its cell at step t is cbase + istep * t, for t - t_lo in [0, nx)
        const int jp = g.tj * DOS_TJ + jj, kp = g.tk * DOS_TK + kk;
        const bool valid = jp < ny && kp < nz;
        const int j = (o & 2) ? ny - 1 - jp : jp;
        const int k = (o & 4) ? nz - 1 - kp : kp;
        const int istep = (o & 1) ? -1 : 1;
        const long long cbase = ((long long)k * ny + j) * nx + ((o & 1) ? nx - 1 : 0) - (long long)istep * skew;
        const int t_lo = valid ? skew : BIG;

        if (tick) {
            // ------- feeder ("tick") warp: tile-inflow faces, material ids, step counter -------
            // Copies the faces the upwind tiles have published (waiting for the service warp's word when they
            // are not there yet), stages the material ids three steps ahead, and after every barrier tells the
            // service warp how many steps are complete. Its CTA-scope release is cheap because its own global
            // traffic is light; the same release from an aux or compute thread would wait for that warp's
            // outstanding red.global / st.global round trips to L2 on every step.
            const int n_fops = 3 * A;
            const LoadOp op0 = make_op<MP, LL>(32 * MV + (lane < n_fops ? lane : 0), p, g, s_q, s_fin);
            const bool op0_on = lane < n_fops, more_ops = n_fops > 32;
            const uint8_t *mat_p = p.mat + cbase + 3 * istep;            // material of step t + 3
            const unsigned mat_w = smem_addr(s_mat + lane);
            auto mat_of = [&](int s, const uint8_t *q) -> int {
                return ((unsigned)(s - t_lo) < (unsigned)nx) ? min((int)__ldg(q), p.n_mat - 1) : 0;
            };
            __syncthreads();                          // S2: s_done, s_allowed in place
            int allowed_c = -1;
            auto issue_one = [&](const LoadOp &d, int tau) {
                const int s = tau + DF;
                if (s >= d.lo && s <= d.hi) {
                    while (allowed_c < s) {           // wait until the upwind tiles have published step s
                        allowed_c = ld_acquire_cta(a_allowed);
                        if (allowed_c < s) __nanosleep(DOS_POLL_NS);
                    }
                    cp_async16(d.dst0 + (s & d.mask) * d.dslot, d.src0 + (long long)s * d.sstep);
                }
            };
            auto issue_round = [&](int tau) {         // round tau fetches the tile-inflow faces of step tau + DF
                if (op0_on) issue_one(op0, tau);
                if (more_ops)
                    for (int f = lane + 32; f < n_fops; f += 32) issue_one(make_op<MP, LL>(32 * MV + f, p, g, s_q, s_fin), tau);
                cp_async_commit();
            };
            // flag-in-data mode: the pairs of step s are requested one step before they are checked (two 16-byte loads per
            // lane, kept in registers), checked -- and re-read until every pair the step needs carries this launch's
            // epoch -- then their values go to the ring slot. A pair is needed if its upwind lane is inside the mesh and
            // active at that diagonal (the others are never written).
            const unsigned ep = (unsigned)p.epoch;
            uint4 ra = make_uint4(0, 0, 0, 0), rb = ra;
            bool req = false;
            auto ll_request = [&](int s) {
                req = op0_on && s >= op0.lo && s <= op0.hi;
                if (req) {
                    const float *sp = op0.src0 + (long long)s * op0.sstep;
                    ra = ld_pairs(sp); rb = ld_pairs(sp + 4);
                }
            };
            auto ll_complete = [&](int s) {
                if (!req) return;
                const bool n0 = op0.e0 + 0 < op0.nval && (unsigned)(s - op0.e0 - 0) < (unsigned)nx;
                const bool n1 = op0.e0 + 1 < op0.nval && (unsigned)(s - op0.e0 - 1) < (unsigned)nx;
                const bool n2 = op0.e0 + 2 < op0.nval && (unsigned)(s - op0.e0 - 2) < (unsigned)nx;
                const bool n3 = op0.e0 + 3 < op0.nval && (unsigned)(s - op0.e0 - 3) < (unsigned)nx;
                const float *sp = op0.src0 + (long long)s * op0.sstep;
                int spins = 0;
                while ((n0 && ra.y != ep) || (n1 && ra.w != ep) || (n2 && rb.y != ep) || (n3 && rb.w != ep)) {
                    if (++spins > DOS_SPIN_LIMIT) { atomicExch(p.abort_flag, 1); break; }      // watchdog, as the service warp's
                    if ((spins & 255) == 0 && ld_relaxed(p.abort_flag)) break;
                    ra = ld_pairs(sp); rb = ld_pairs(sp + 4);
                }
                sts_v4(op0.dst0 + (s & op0.mask) * op0.dslot,
                       make_float4(__uint_as_float(ra.x), __uint_as_float(ra.z), __uint_as_float(rb.x), __uint_as_float(rb.z)));
            };
            if (LL) {
                ll_request(0); ll_complete(0); ll_request(1);
            } else {
                for (int tau = -DF; tau < 0; ++tau) issue_round(tau);
            }
            sts_s32(mat_w, mat_of(0, mat_p - 3 * istep));
            sts_s32(mat_w + 128, mat_of(1, mat_p - 2 * istep));
            int reg_m = mat_of(2, mat_p - istep);
            cp_async_wait<DF - 1>();
            bar_compute(NB);                          // S3: step 0's staged data visible to every warp
#pragma unroll 1
            for (int t = 0; t < T; ++t) {
                if (LL) { ll_complete(t + 1); ll_request(t + 2); }
                else issue_round(t);
                sts_s32(mat_w + ((t + 2) & 3) * 128, reg_m);
                reg_m = mat_of(t + 3, mat_p);
                mat_p += istep;
                cp_async_wait<DF - 1>();              // step t + 1's faces complete (this thread's copies)
                bar_compute(NB);                      // B_t: ... visible to all; every face store of step t precedes it
                if (lane == 0) st_release_cta(a_done, t + 1);
            }
            continue;
        }

        if (aux) {
            // ---------------- aux warps: staging, material ids, D2M of the previous step ----------------
            const int xw = warp - NW, xt = tid - NW * 32, NXT = NX * 32;
            const int n_ops = 32 * MV;                                   // Q copies; the feeder warp does the faces
            const LoadOp op0 = make_op<MP, LL>(xt < n_ops ? xt : 0, p, g, s_q, s_fin);
            const LoadOp op1 = make_op<MP, LL>(xt + NXT < n_ops ? xt + NXT : 0, p, g, s_q, s_fin);
            const bool op0_on = xt < n_ops, op1_on = xt + NXT < n_ops, more_ops = n_ops > 2 * NXT;
            float *phi_p = p.phi + (cbase - istep) * MP;                 // moments of the cell of step t - 1
            const int phi_inc = istep * MP;
            const unsigned psi_r = smem_addr(s_psi + lane), d2m_a = smem_addr(s_d2m);
            const int psi_slot = A * 32 * 4;
            __syncthreads();                          // S2: octant tables in place
            auto issue_one = [&](const LoadOp &d, int tau) {
                const int s = tau + DQ;
                if (s >= d.lo && s <= d.hi) cp_async16(d.dst0 + (s & d.mask) * d.dslot, d.src0 + (long long)s * d.sstep);
            };
            auto issue_round = [&](int tau) {         // round tau fetches the source moments of step tau + DQ
                if (op0_on) issue_one(op0, tau);
                if (op1_on) issue_one(op1, tau);
                if (more_ops)
                    for (int op = xt + 2 * NXT; op < n_ops; op += NXT) issue_one(make_op<MP, LL>(op, p, g, s_q, s_fin), tau);
                cp_async_commit();
            };
            for (int tau = -DQ; tau < 0; ++tau) issue_round(tau);
            cp_async_wait<DQ - 1>();
            bar_compute(NB);                          // S3: step 0's staged data visible to every warp

#pragma unroll 1
            for (int t = 0; t < T; ++t) {
                issue_round(t);
                // D2M of step t - 1: sum over all angles of the octant, one red per (cell, 4 moments)
                if (t > 0 && (unsigned)(t - 1 - t_lo) < (unsigned)nx) {
                    const unsigned ps = psi_r + ((t - 1) & 1) * psi_slot;
                    for (int v = xw; v < MV; v += NX) {
                        const unsigned dp = d2m_a + 16 * v;
                        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 5
                        for (int a = 0; a < A; ++a) {
                            const float psi = lds_f32(ps + a * 128);
                            const float4 d = lds_v4(dp + a * (MP * 4));
                            acc.x = fmaf(d.x, psi, acc.x);
                            acc.y = fmaf(d.y, psi, acc.y);
                            acc.z = fmaf(d.z, psi, acc.z);
                            acc.w = fmaf(d.w, psi, acc.w);
                        }
                        red_add_v4(phi_p + 4 * v, acc);
                    }
                }
                phi_p += phi_inc;
                cp_async_wait<DQ - 1>();              // step t + 1's staged data (issued DQ rounds ago) complete; the younger rounds stay in flight
                bar_compute(NB);                      // B_t: ... and visible to all
            }
            if ((unsigned)(T - 1 - t_lo) < (unsigned)nx) {
                const unsigned ps = psi_r + ((T - 1) & 1) * psi_slot;
                for (int v = xw; v < MV; v += NX) {
                    const unsigned dp = d2m_a + 16 * v;
                    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
                    for (int a = 0; a < A; ++a) {
                        const float psi = lds_f32(ps + a * 128);
                        const float4 d = lds_v4(dp + a * (MP * 4));
                        acc.x = fmaf(d.x, psi, acc.x);
                        acc.y = fmaf(d.y, psi, acc.y);
                        acc.z = fmaf(d.z, psi, acc.z);
                        acc.w = fmaf(d.w, psi, acc.w);
                    }
                    red_add_v4(phi_p + 4 * v, acc);
                }
            }
            continue;
        }

        // ---------------- compute warps: M2D, diamond difference, face hand-off ----------------
        constexpr bool REGC = AG * MP <= 48;          // M2D coefficients of this warp's angles in registers
        const int a0 = warp * AG;
        const bool in_y = jj == 0, in_z = kk == 0;
        const bool has_y = g.has_y, has_z = g.has_z;
        const bool store_y = valid && jj == DOS_TJ - 1 && g.tj < p.ntj - 1;
        const bool store_z = valid && kk == DOS_TK - 1 && g.tk < p.ntk - 1;
        // running pointers, advanced once per step
        constexpr int lls = LL ? 2 : 1;             // floats per face value: (value, epoch) pairs in flag-in-data mode
        const unsigned ep = (unsigned)p.epoch;
        float *fy_st = p.fy + ((long long)((size_t)g.id * fstride_y) + kk + ((long long)(1 - DOS_TJ) * A + a0) * DOS_TK) * lls;
        float *fz_st = p.fz + ((long long)((size_t)g.id * fstride_z) + jj + ((long long)(1 - DOS_TK) * A + a0) * DOS_TJ) * lls;
        const int fy_inc = A * DOS_TK * lls, fz_inc = A * DOS_TJ * lls;
        const unsigned fin_y = smem_addr(s_fin + a0 * FINW + kk), fin_z = smem_addr(s_fin + a0 * FINW + DOS_TK + jj);
        const unsigned psi_w = smem_addr(s_psi + a0 * 32 + lane);
        const unsigned q_row = smem_addr(s_q + lane * MPS);
        const unsigned rden_a = smem_addr(s_rden + a0), sig_a = smem_addr(s_sig), mat_r = smem_addr(s_mat + lane);
        const unsigned m2d_a = smem_addr(s_m2d + a0 * MP);
        const int fin_slot = A * FINW * 4, psi_slot = A * 32 * 4, A4 = A * 4;

        float cm[REGC ? AG * MP : 1];
        float ccx[AG], ccy[AG], ccz[AG];
        __syncthreads();                              // S2: octant tables, s_done, s_allowed in place
        if (REGC) {
#pragma unroll
            for (int r = 0; r < AG; ++r)
#pragma unroll
                for (int e = 0; e < MP; ++e) cm[REGC ? r * MP + e : 0] = s_m2d[(a0 + r) * MP + e];
        }
#pragma unroll
        for (int r = 0; r < AG; ++r) {
            ccx[r] = s_cdd[(a0 + r) * 4 + 0]; ccy[r] = s_cdd[(a0 + r) * 4 + 1]; ccz[r] = s_cdd[(a0 + r) * 4 + 2];
        }
        float px[AG], oy[AG], oz[AG];
#pragma unroll
        for (int r = 0; r < AG; ++r) px[r] = oy[r] = oz[r] = 0.f;
        bar_compute(NB);                              // S3: step 0's staged data visible

#pragma unroll 1
        for (int t = 0; t < T; ++t) {
            // moment-to-discrete for this lane's cell, AG angles; four partial sums keep the FMA chains short
            const bool act = (unsigned)(t - t_lo) < (unsigned)nx;
            const int m0 = lds_s32(mat_r + (t & 3) * 128);
            float q[AG];
            {
                float part[AG][4];
#pragma unroll
                for (int r = 0; r < AG; ++r) part[r][0] = part[r][1] = part[r][2] = part[r][3] = 0.f;
                const unsigned qs = q_row + (t & (RQ - 1)) * (32 * MPS * 4);
#pragma unroll
                for (int v = 0; v < MV; ++v) {
                    const float4 qv = lds_v4(qs + 16 * v);
#pragma unroll
                    for (int r = 0; r < AG; ++r) {
                        float4 c;
                        if (REGC) c = make_float4(cm[REGC ? r * MP + 4 * v : 0], cm[REGC ? r * MP + 4 * v + 1 : 0],
                                                  cm[REGC ? r * MP + 4 * v + 2 : 0], cm[REGC ? r * MP + 4 * v + 3 : 0]);
                        else c = lds_v4(m2d_a + (r * MP + 4 * v) * 4);
                        part[r][v & 3] = fmaf(c.x, qv.x, fmaf(c.y, qv.y, fmaf(c.z, qv.z, fmaf(c.w, qv.w, part[r][v & 3]))));
                    }
                }
#pragma unroll
                for (int r = 0; r < AG; ++r) q[r] = (part[r][0] + part[r][1]) + (part[r][2] + part[r][3]);
            }
            // inflow, diamond difference, outflow
            const unsigned fslot = (t & (RF - 1)) * fin_slot;
            const unsigned pso = psi_w + (t & 1) * psi_slot;
            const unsigned rd = rden_a + m0 * A4;
            const bool first_x = t == t_lo;
#pragma unroll
            for (int r = 0; r < AG; ++r) {
                float yin = __shfl_up_sync(0xffffffffu, oy[r], 1);
                float zin = __shfl_up_sync(0xffffffffu, oz[r], DOS_TJ);
                if (in_y) yin = has_y ? lds_f32(fin_y + fslot + r * (FINW * 4)) : 0.f;    // tile inflow or vacuum
                if (in_z) zin = has_z ? lds_f32(fin_z + fslot + r * (FINW * 4)) : 0.f;
                float pc = 0.f;
                if (act) {
                    const float ix = first_x ? 0.f : px[r];
                    const float num = fmaf(ccx[r], ix, fmaf(ccy[r], yin, fmaf(ccz[r], zin, q[r])));
                    pc = num * lds_f32(rd + 4 * r);
                    float ox = 2.f * pc - ix, oyr = 2.f * pc - yin, ozr = 2.f * pc - zin;
                    if (fminf(ox, fminf(oyr, ozr)) < 0.f)
                        dd_fixup(pc, ox, oyr, ozr, q[r], lds_f32(sig_a + 4 * m0), ccx[r], ccy[r], ccz[r], ix, yin, zin);
                    px[r] = ox; oy[r] = oyr; oz[r] = ozr;
                    if (lls == 2) {
                        if (store_y) st_pair(fy_st + r * (2 * DOS_TK), oyr, ep);
                        if (store_z) st_pair(fz_st + r * (2 * DOS_TJ), ozr, ep);
                    } else {
                        if (store_y) __stcg(fy_st + r * DOS_TK, oyr);
                        if (store_z) __stcg(fz_st + r * DOS_TJ, ozr);
                    }
                }
                sts_f32(pso + r * 128, pc);
            }
            fy_st += fy_inc; fz_st += fz_inc;
            bar_compute(NB);                          // B_t
        }
    }
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side: choice of angles per warp, occupancy-sized persistent grid, template dispatch
// ------------------------------------------------------------------------------------------------
typedef void (*sweep_fn)(const Sweep2Args);

// variant 0: up to 16 warps, 1 CTA per SM; 1: up to 24 warps; 2: up to 16 warps capped at 64 registers so that two
// CTAs share an SM (MP <= 16 only) -- on meshes with many more work items than SMs the second CTA fills the other's
// barrier and latency stalls (config 4: measured in DESIGN.md section 6)
template <int MP, int AG>
static sweep_fn pick_var(int var, bool ll)
{
    if (ll) return (var == 0 && MP <= 16) ? sweep_kernel<(MP <= 16 ? MP : 4), AG, 512, 1, true> : nullptr;
    if (var == 1) return sweep_kernel<MP, AG, 768, 1, false>;
    if (var == 2) return MP <= 16 ? sweep_kernel<(MP <= 16 ? MP : 4), AG, 512, 2, false> : nullptr;
    return sweep_kernel<MP, AG, 512, 1, false>;
}

template <int MP>
static sweep_fn pick_ag(int ag, int var, bool ll)
{
    switch (ag) {
        case 1: return pick_var<MP, 1>(var, ll);
        case 2: return pick_var<MP, 2>(var, ll);
        case 3: return pick_var<MP, 3>(var, ll);
        case 4: return pick_var<MP, 4>(var, ll);
    }
    return nullptr;
}

// two_per_sm: 1: variant 2 from 4 work items per SM, 2: whenever there are more items than SMs, 0: never (per context)
// ll: the flag-in-data instance (one CTA per SM, P0..P3, at most 10 angles per CTA), nullptr where there is none
static sweep_fn pick(int L, int ag, int per_oct, int n_aux, int n_items, int two_per_sm, bool ll = false)
{
    const int warps = per_oct / ag + n_aux + 2, MP = dos_mpad(L);
    int sms = 148, dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int var = warps > 16 ? 1 : ((two_per_sm && MP <= 16 && (two_per_sm == 2 ? n_items > sms : n_items >= 4 * sms)) ? 2 : 0);
    switch (MP) {
        case 4: return pick_ag<4>(ag, var, ll && 3 * per_oct <= 32);
        case 12: return pick_ag<12>(ag, var, ll && 3 * per_oct <= 32);
        case 16: return pick_ag<16>(ag, var, ll && 3 * per_oct <= 32);
        case 28: return ll ? nullptr : pick_ag<28>(ag, var, false);
        case 36: return ll ? nullptr : pick_ag<36>(ag, var, false);
    }
    return nullptr;
}

static size_t sweep_smem(int L, int per_oct, int n_mat)
{
    const int MP = dos_mpad(L), MPS = mps_of(MP), A = per_oct;
    const size_t floats = (size_t)RQ * 32 * MPS + (size_t)RF * A * FINW + (size_t)2 * A * 32 + (size_t)2 * A * MP +
                          (size_t)4 * A + (size_t)n_mat * A + ((n_mat + 3) & ~3) + 4 * 32 + 4;
    return sizeof(float) * floats;
}

// Angles per warp AG (1..4, must divide the octant's angle count A; the CTA has A/AG compute warps and
// one service warp, at most 21 warps). Default: the smallest AG with at most 12 compute warps -- few
// angles per warp keep the per-step dependent chain short (S2: 1x1, S4: 3x1, S6: 6x1, S8: 10x1,
// S12: 7x3, S16: 12x3). `prefer` > 0 overrides when it is admissible.
// Aux warps (staging + D2M): one per 4-moment quad when the CTA then stays within 24 warps, else fewer
// (each takes several quads). `prefer` > 0 overrides (clamped to [1, MP/4]).
int dos_sweep_ffma_aux_warps(int per_oct, int L, int ag, int prefer)
{
    const int mv = dos_mpad(L) / 4, nw = per_oct / ag;
    if (prefer >= 1) return prefer < mv ? prefer : mv;
    int nx = mv;
    while (nx > 1 && nw + nx + 2 > 24) nx = (nx + 1) / 2;
    return nx;
}

int dos_sweep_ffma_angles_per_warp(int per_oct, int L, int prefer)
{
    (void)L;
    if (prefer >= 1 && prefer <= 4 && per_oct % prefer == 0 && per_oct / prefer <= (prefer <= 2 ? 20 : 12)) return prefer;
    for (int ag = 1; ag <= 4; ++ag)
        if (per_oct % ag == 0 && per_oct / ag <= 12) return ag;
    for (int ag = 1; ag <= 2; ++ag)
        if (per_oct % ag == 0 && per_oct / ag <= 20) return ag;
    return 0;
}

cudaError_t dos_sweep_ffma_grid(int L, int ag, int n_aux, int per_oct, int n_mat, int n_items, int two_per_sm, int *grid_out)
{
    sweep_fn f = pick(L, ag, per_oct, n_aux, n_items, two_per_sm);
    if (!f) return cudaErrorInvalidValue;
    const size_t smem = sweep_smem(L, per_oct, n_mat);
    cudaError_t e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (sweep_fn fl = pick(L, ag, per_oct, n_aux, n_items, two_per_sm, true))       // same shape, same grid
        if ((e = cudaFuncSetAttribute(fl, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
    int dev = 0, sms = 0, per_sm = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    const int threads = (per_oct / ag + n_aux + 2) * 32;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, f, threads, smem)) != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    // Persistent CTAs: every resident CTA pulls items until the queue is empty. All CTAs of the grid
    // must be co-resident only for speed, not for progress: an item never waits on a later item.
    int g = sms * per_sm;
    *grid_out = g < n_items ? g : n_items;
    return cudaSuccess;
}

cudaError_t dos_launch_sweep_ffma(const Sweep2Args &a, int L, int ag, int grid, int two_per_sm, cudaStream_t s)
{
    sweep_fn f = pick(L, ag, a.per_oct, a.n_aux, a.n_items, two_per_sm);
    if (!f) return cudaErrorInvalidValue;
    if (a.ll) {      // the caller's buffers hold pairs and an epoch is set: take the flag-in-data instance where there is one
        if (sweep_fn fl = pick(L, ag, a.per_oct, a.n_aux, a.n_items, two_per_sm, true)) f = fl;
    }
    const size_t smem = sweep_smem(L, a.per_oct, a.n_mat);
    f<<<grid, (a.n_warps + a.n_aux + 2) * 32, smem, s>>>(a);
    return cudaGetLastError();
}
