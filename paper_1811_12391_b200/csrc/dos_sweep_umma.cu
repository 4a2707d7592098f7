// dos_sweep_umma.cu -- the S_N transport sweep (eq. 2-3) for one group and one source iteration on
// the Blackwell tensor-memory path: moment-to-discrete (a5) and discrete-to-moment (a7) are tcgen05.mma (kind::tf32,
// 3xTF32 split, fp32 accumulate in TMEM), the source moments arrive by bulk asynchronous copies (TMA unit) that complete
// on mbarriers, and every hand-off inside the CTA is an mbarrier ring: there is no CTA-wide barrier in the step loop.
// The diamond-difference cell update with set-to-zero fixup and rebalance (a6; north_star; R3, R11, R12) runs
// in ordinary warps between the two contractions. DESIGN.md section 6 has the measurements behind the shape.
//
//   work item   (octant quad, tile of 8 x 4 (j,k) columns in octant-local indices), whole x range: the CTA sweeps the
//               SAME local tile for the 4 octants of a quad (xi > 0 or xi < 0) at once. The 4 octants are the 4
//               32-lane quarters of the 128-row UMMA tile, and a warp may only touch the TMEM lanes of quarter
//               (warp % 4): so warp % 4 = octant, everywhere.
//   row         (octant q, lane) = TMEM lane 32 q + lane = that octant's (j,k) column `lane` of the tile, at cell
//               x_local = step - (jj + kk): the KBA wavefront inside the warp, as in dos_sweep_ffma.cu.
//   M2D         D_q[row][angle] = sum_lm A[row][lm] B[lm][angle], A = the row's source moments with the octant's
//               mirror signs applied (Y_lm of a mirrored direction is +-Y_lm: the sign depends on (l,m) and the mirror
//               only), split into TF32 hi + lo by the `split` warps and written to shared memory in the UMMA K-major
//               core-matrix layout; B = (2l+1) Y_lm of octant 0's angles, pre-split on the host. 3 terms
//               (lo*hi, hi*lo, hi*hi) x K/8 instructions, issued by one thread, accumulator ring in TMEM.
//   cell update compute warp (octant q, angle group g) reads its AG columns of D_q straight from TMEM (tcgen05.ld),
//               takes the y/z inflow from the neighbouring lanes by shuffle (or from the staged tile-inflow faces),
//               and writes psi_c, split into hi + lo, back to TMEM (tcgen05.st) as the A operand of
//   D2M         D_phi[row][lm] = sum_a psi[row][a] w_a Y_lm(a) (A from TMEM, B from shared memory), after which the
//               `epilogue` warps read D_phi (tcgen05.ld), apply the mirror signs and red.global.add.v4 into phi.
//   tile faces  as in dos_sweep_ffma.cu: outflow of the tile's last j / k lanes goes to an L2-resident buffer indexed
//               by wavefront diagonal, published every `chunk` steps by the service warp (st.release.gpu), acquired by
//               the downwind CTA's service warp, staged by its feeder warp with bulk copies.
// The angular flux never leaves registers / tensor memory.
#include <utility>

#include "dos_internal.h"
#include "dos_sm100.cuh"

namespace {

using namespace sm100;

constexpr int RAW = 4;       // ring of staged source-moment rows (steps)
constexpr int LA = 3;        // steps between issuing a row's bulk copy and using it
constexpr int ASL = 2;       // ring of split A operands (hi, lo) in shared memory
constexpr int DQS = 4;       // ring of M2D accumulators in TMEM
constexpr int PSL = 2;       // ring of psi operands (hi, lo) in TMEM
constexpr int DPS = 2;       // ring of D2M accumulators in TMEM
constexpr int RFU = 4;       // ring of staged tile-inflow faces (steps)
constexpr int BIG = 1 << 30;
constexpr int WAIT_LIMIT = 1 << 24;     // sleeping polls (>= 64 ns each: seconds) before a wait declares the launch stuck
#ifndef DOS_UMMA_TRACE
#define DOS_UMMA_TRACE 0      // measurement builds only: SM-clock timeline of one work item into the face buffer's tail
#endif
#if DOS_UMMA_TRACE
#define TRACE(ev) do { if (trace_on && lane == 0 && t >= 100 && t < 164) trace_buf[((warp * 64 + (t - 100)) * 8) + (ev)] = clock64(); } while (0)
#else
#define TRACE(ev) do { } while (0)
#endif
#ifndef DOS_UMMA_ABL
#define DOS_UMMA_ABL 0        // measurement builds only: bit 0 no source-moment copies, 1 no reds, 2 no MMAs, 3 no cell update
#endif

__device__ __forceinline__ int ld_relaxed_gpu(const int *p)
{
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ void st_release_gpu(int *p, int v) { asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory"); }
__device__ __forceinline__ void st_release_cta(int *p, int v)
{
    asm volatile("st.release.cta.shared.s32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
__device__ __forceinline__ int ld_acquire_cta(const int *p)
{
    int v;
    asm volatile("ld.acquire.cta.shared.s32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ void red_add_v4(float *p, float a, float b, float c, float d)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

// Bounded wait on an mbarrier phase. A waiting warp must not spend issue slots: measured, try_wait returns within
// ~50 cycles whether or not it carries a suspend-time hint, and twelve helper warps polling back to back issued more
// instructions than the sixteen compute warps doing the work. So: one poll, then sleep between polls.
// A hand-off that never arrives must not hang the GPU: the waiter sets the CTA's and the launch's abort flags and
// everything drains with invalid results (dos_check then reports DOS_ERR_CUDA).
__device__ __forceinline__ void wait_bar(uint64_t *bar, unsigned parity, int *s_abort, int *g_abort, unsigned sleep_ns = 64)
{
    if (mbar_try_wait(bar, parity)) return;
#pragma unroll 1
    for (int spins = 0; spins < WAIT_LIMIT; ++spins) {
        __nanosleep(sleep_ns);
        if (mbar_try_wait(bar, parity)) return;
        if ((spins & 1023) == 1023 && *(volatile int *)s_abort) return;
    }
    *(volatile int *)s_abort = 1;
    atomicExch(g_abort, 1);
}

// Slow path of the cell update: at least one extrapolated outflow was negative. Faces found negative are pinned to
// zero together, the balance is re-solved, and the pinned set only grows (R12).
__device__ __forceinline__ void dd_fixup(float &pc, float &ox, float &oy, float &oz, float q, float st, float cx, float cy, float cz,
                                         float ix, float iy, float iz)
{
    const float hx = cx * ix, hy = cy * iy, hz = cz * iz;
    bool fx = false, fy = false, fz = false;
#pragma unroll 1
    do {
        fx |= ox < 0.f; fy |= oy < 0.f; fz |= oz < 0.f;
        const float num = q + (fx ? 0.5f * hx : hx) + (fy ? 0.5f * hy : hy) + (fz ? 0.5f * hz : hz);
        const float den = st + (fx ? 0.f : cx) + (fy ? 0.f : cy) + (fz ? 0.f : cz);
        pc = __fdividef(num, den);
        ox = fx ? 0.f : 2.f * pc - ix;
        oy = fy ? 0.f : 2.f * pc - iy;
        oz = fz ? 0.f : 2.f * pc - iz;
    } while (fminf(ox, fminf(oy, oz)) < 0.f);
}

// hi = x rounded to TF32 (round half away from zero on the bit pattern; inputs are finite), lo = x - hi (exact in
// fp32; the tensor core reads its leading 11 bits: an error <= 2^-22 |x|)
__device__ __forceinline__ void tf32_split(float x, float &hi, float &lo)
{
    hi = __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
    lo = x - hi;
}

__host__ __device__ constexpr int umma_reg_compute(int ng) { return ng == 4 ? 96 : 120; }
__host__ __device__ constexpr int umma_reg_helper(int) { return 40; }

struct Geom {          // one octant's (j,k) column of this lane
    bool valid;
    int t_lo;          // first active step (skew), BIG if the column is outside the mesh
    long long cbase;   // cell at step t: cbase + istep * t
    int istep;
};

__device__ __forceinline__ Geom make_geom(const SweepUArgs &p, int o, int tj, int tk, int lane)
{
    const int jj = lane & (DOS_TJ - 1), kk = lane / DOS_TJ, skew = jj + kk;
    const int jp = tj * DOS_TJ + jj, kp = tk * DOS_TK + kk;
    Geom g;
    g.valid = jp < p.ny && kp < p.nz;
    const int j = (o & 2) ? p.ny - 1 - jp : jp, k = (o & 4) ? p.nz - 1 - kp : kp;
    g.istep = (o & 1) ? -1 : 1;
    g.cbase = g.valid ? ((long long)k * p.ny + j) * p.nx + ((o & 1) ? p.nx - 1 : 0) - (long long)g.istep * skew : 0;
    g.t_lo = g.valid ? skew : BIG;
    return g;
}

// Epilogue of one row: D_phi columns [C0, MP) -> mirror signs -> phi[cell][C0..MP) by red.global.add.v4, 8 columns at a time.
template <int MP, int C0>
__device__ __forceinline__ void epilogue_row(unsigned taddr, const unsigned *sgn, float *phi, bool on)
{
    if constexpr (C0 < MP) {
        constexpr int N = MP - C0 < 8 ? MP - C0 : 8;
        float v[N];
        tmem_ld_n<N>(taddr + C0, v);
        tmem_wait_ld();
        if (on && !(DOS_UMMA_ABL & 2)) {
#pragma unroll
            for (int e = 0; e < N; e += 4) {
                const uint4 s = *reinterpret_cast<const uint4 *>(sgn + C0 + e);
                red_add_v4(phi + C0 + e, __uint_as_float(__float_as_uint(v[e]) ^ s.x), __uint_as_float(__float_as_uint(v[e + 1]) ^ s.y),
                           __uint_as_float(__float_as_uint(v[e + 2]) ^ s.z), __uint_as_float(__float_as_uint(v[e + 3]) ^ s.w));
            }
        }
        epilogue_row<MP, C0 + N>(taddr, sgn, phi, on);
    }
}

// Split warp, one row of NQ float4: stage (cp.async) and convert (mirror signs, TF32 hi / lo, UMMA core-matrix layout).
template <int NQ>
__device__ __forceinline__ void split_issue(float *dst, const float *src)
{
#pragma unroll
    for (int c = 0; c < NQ; ++c) cp_async16(dst + 4 * c, src + 4 * c);
}
template <int NQ>
__device__ __forceinline__ void split_row(const float4 *src, const unsigned *sgn, float4 *dh, float4 *dl, bool on)
{
#pragma unroll
    for (int b = 0; b < NQ; b += 3) {                 // 3 float4 in flight: the helper warps live in 40 registers
        float4 x[3];
#pragma unroll
        for (int c = 0; c < 3; ++c)
            if (b + c < NQ) x[c] = on ? src[b + c] : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int c = 0; c < 3; ++c)
            if (b + c < NQ) {
                const uint4 s4 = *reinterpret_cast<const uint4 *>(sgn + 4 * (b + c));
                float4 h, l;
                tf32_split(__uint_as_float(__float_as_uint(x[c].x) ^ s4.x), h.x, l.x);
                tf32_split(__uint_as_float(__float_as_uint(x[c].y) ^ s4.y), h.y, l.y);
                tf32_split(__uint_as_float(__float_as_uint(x[c].z) ^ s4.z), h.z, l.z);
                tf32_split(__uint_as_float(__float_as_uint(x[c].w) ^ s4.w), h.w, l.w);
                dh[(b + c) * 8] = h;
                dl[(b + c) * 8] = l;
            }
    }
}

// Warp roles (NG compute warps per octant, AG angles each):
//   [0, 4 NG)            compute: octant q = warp % 4, angle group g = warp / 4
//   [4 NG, 4 NG + 4)     split:   octant q; bulk copies of the rows' source moments, mirror signs, TF32 split
//   [.. + 4, .. + 8)     epilogue: octant q; D_phi -> phi
//   .. + 8               M2D issuer (one elected lane)      .. + 9   D2M issuer
//   .. + 10              feeder (tile-inflow faces)         .. + 11  service (global hand-off flags)
template <int AG, int NG>
__global__ void __launch_bounds__((4 * NG + 12) * 32, 1) sweep_umma_kernel(const SweepUArgs p)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int A = p.per_oct, MP = p.MP, KP = (MP + 7) & ~7, NCH = KP / 4, A8 = (A + 7) & ~7, NAP = (A + 15) & ~15, NMP = (MP + 15) & ~15;
    constexpr int NCW = 4 * NG;
    // ---- shared memory carve-up (every piece a multiple of 128 bytes) ----
    unsigned char *sp = smem_raw;
    auto carve = [&](size_t bytes) { unsigned char *r = sp; sp += (bytes + 127) & ~(size_t)127; return r; };
    float *s_raw = reinterpret_cast<float *>(carve((size_t)RAW * 128 * MP * 4));                 // [RAW][128 rows][MP]
    float *s_a = reinterpret_cast<float *>(carve((size_t)ASL * 2 * 16 * NCH * 128));            // [ASL][hi,lo][16][NCH][8][4]
    float *s_bm = reinterpret_cast<float *>(carve((size_t)2 * (NAP / 8) * NCH * 128));          // [hi,lo][NAP/8][NCH][8][4]
    float *s_bd = reinterpret_cast<float *>(carve((size_t)2 * (NMP / 8) * (A8 / 4) * 128));     // [hi,lo][NMP/8][A8/4][8][4]
    float *s_finy = reinterpret_cast<float *>(carve((size_t)RFU * 4 * A * DOS_TK * 4));         // [RFU][4][A][TK]
    float *s_finz = reinterpret_cast<float *>(carve((size_t)RFU * 4 * A * DOS_TJ * 4));         // [RFU][4][A][TJ]
    float *s_cdd = reinterpret_cast<float *>(carve((size_t)A * 16));                            // [A][4]
    float *s_rden = reinterpret_cast<float *>(carve((size_t)p.n_mat * A * 4));                  // [n_mat][A]
    float *s_sig = reinterpret_cast<float *>(carve((size_t)p.n_mat * 4));
    unsigned *s_sign = reinterpret_cast<unsigned *>(carve((size_t)8 * MP * 4));                 // [8 octants][MP] 0 or 0x80000000
    uint64_t *bars = reinterpret_cast<uint64_t *>(carve(64 * 8));
    int *s_prog = reinterpret_cast<int *>(carve(32 * 4));                                       // [NCW] steps finished per compute warp
    uint64_t *raw_full = bars;            // [RAW][4]
    uint64_t *a_full = bars + 16;         // [ASL]
    uint64_t *a_empty = bars + 18;
    uint64_t *q_full = bars + 20;         // [DQS]
    uint64_t *q_empty = bars + 24;
    uint64_t *psi_full = bars + 28;       // [PSL]
    uint64_t *psi_empty = bars + 30;
    uint64_t *phi_full = bars + 32;       // [DPS]
    uint64_t *phi_empty = bars + 34;
    uint64_t *fin_full = bars + 36;       // [RFU]
    __shared__ int s_item, s_allowed, s_abort;
    __shared__ unsigned s_tmem;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, q = warp & 3;
    const bool is_compute = warp < NCW, is_split = warp >= NCW && warp < NCW + 4, is_epi = warp >= NCW + 4 && warp < NCW + 8;
    const bool is_m2d = warp == NCW + 8, is_d2m = warp == NCW + 9, is_feed = warp == NCW + 10, is_service = warp == NCW + 11;
    const int nx = p.nx, T = nx + DOS_SKEW;
    const size_t fstride_y = (size_t)(nx + DOS_FACE_PAD) * A * DOS_TK, fstride_z = (size_t)(nx + DOS_FACE_PAD) * A * DOS_TJ;

    // ---- one-time set-up ----
    for (int i = tid; i < 2 * (NAP / 8) * NCH * 32; i += blockDim.x) s_bm[i] = p.bm2d[i];
    for (int i = tid; i < 2 * (NMP / 8) * (A8 / 4) * 32; i += blockDim.x) s_bd[i] = p.bd2m[i];
    for (int i = tid; i < ASL * 2 * 16 * NCH * 32; i += blockDim.x) s_a[i] = 0.f;      // K padding columns stay zero for ever
    for (int i = tid; i < A * 4; i += blockDim.x) s_cdd[i] = p.cdd[i];
    for (int i = tid; i < p.n_mat * A; i += blockDim.x) s_rden[i] = 1.f / (p.sig_t[i / A] + p.cdd[(i % A) * 4 + 3]);
    for (int i = tid; i < p.n_mat; i += blockDim.x) s_sig[i] = p.sig_t[i];
    for (int i = tid; i < 8 * MP; i += blockDim.x) s_sign[i] = p.signs[i];
    if (tid == 0) {
        for (int i = 0; i < 16; ++i) mbar_init(&raw_full[i], 32);
        for (int i = 0; i < ASL; ++i) { mbar_init(&a_full[i], 4); mbar_init(&a_empty[i], 1); }
        for (int i = 0; i < DQS; ++i) { mbar_init(&q_full[i], 1); mbar_init(&q_empty[i], NCW); }
        for (int i = 0; i < PSL; ++i) { mbar_init(&psi_full[i], NCW); mbar_init(&psi_empty[i], 1); }
        for (int i = 0; i < DPS; ++i) { mbar_init(&phi_full[i], 1); mbar_init(&phi_empty[i], 4); }
        for (int i = 0; i < RFU; ++i) mbar_init(&fin_full[i], 1);
        s_abort = 0;
        mbar_init_fence();
    }
    if (warp == 0) tmem_alloc_512(&s_tmem);
    fence_proxy_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const unsigned tm = s_tmem;
    // TMEM columns: [0, DQS*NAP) M2D accumulators | psi operands [PSL][hi A8 | lo A8] | [DPS][NMP] D2M accumulators
    const unsigned tm_dq = tm, tm_psi = tm + DQS * NAP, tm_dphi = tm_psi + PSL * 2 * A8;
    const unsigned lane_base = (unsigned)(q * 32) << 16;
    if (is_compute) {
        // the K padding columns of the psi operands must be finite (they meet zero rows of B): zero them once
        float z[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        if (warp < 4)
            for (int c = 0; c < PSL * 2 * A8; c += 8) tmem_st<8>(tm_psi + lane_base + c, z);
        tmem_wait_st();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    unsigned gs0 = 0;      // global step counter at the start of the current item (ring slots and phases follow it)
    unsigned fs0 = 0;      // the same for the tile-inflow ring, which only items with an upwind tile use
    // Every role runs its own loop over the work items (so that each role's code lies behind its own setmaxnreg and
    // ptxas can give it its own register budget); all of them meet in the two barriers of next_item().
    int quad = 0, tj = 0, tk = 0, fid = 0;
    bool has_y = false, has_z = false;
#if DOS_UMMA_TRACE
    bool trace_on = false;
    long long *trace_buf = reinterpret_cast<long long *>(p.fz);      // measurement build: the z-face buffer of item 0 is sacrificed
#endif
    auto next_item = [&]() -> bool {
        __syncthreads();                              // every role has drained the previous item
        if (tid == 0) s_item = atomicAdd(p.queue, 1);
        if (tid < NCW) s_prog[tid] = 0;
        __syncthreads();
        const int item = s_item;
        if (item >= p.n_items) return false;
        const int packed = p.items[item];
        quad = packed & 7; tj = (packed >> 3) & 0x3FFF; tk = packed >> 17;
        fid = (quad * p.ntk + tk) * p.ntj + tj;      // hand-off flag of this (quad, tile)
        has_y = tj > 0; has_z = tk > 0;
#if DOS_UMMA_TRACE
        trace_on = item == 601;
#endif
        return true;
    };
    // Register re-allocation (warp roles come in aligned groups of 4 warps, as setmaxnreg requires): the compute warps
    // carry 3 face fluxes per angle plus the cell update's temporaries, the helper warps need little.
    // setmaxnreg re-divides the CTA's OWN register allocation (threads x registers at launch), it cannot draw on the
    // rest of the register file: with more than the launch total the increase blocks for ever. NG = 4: 896 threads x 72 =
    // 16 warps x 96 + 12 x 40; NG = 3: 768 x 80 = 12 x 120 + 12 x 40 (dos_sweep_umma_grid checks the launch count).
    constexpr int REG_C = umma_reg_compute(NG), REG_H = umma_reg_helper(NG);
    constexpr bool REALLOC = NG >= 3;

    if (is_service) {
        if constexpr (REALLOC) setmaxnreg_dec<REG_H>();
        while (next_item()) {
            // ------- service warp: publishes this item's progress, follows the two upwind items' progress -------
            const int *up_y = p.done + (has_y ? fid - 1 : fid), *up_z = p.done + (has_z ? fid - p.ntj : fid);
            int *my_flag = p.done + fid;
            int avail_y = has_y ? 0 : BIG, avail_z = has_z ? 0 : BIG;
            if (lane == 0) s_allowed = (has_y || has_z) ? -1 : BIG;
            __syncthreads();                          // S2
            int published = 0, spins = 0;
            for (;;) {
                int mine = lane < NCW ? ld_acquire_cta(&s_prog[lane]) : BIG;
#pragma unroll
                for (int d = 16; d >= 1; d >>= 1) mine = min(mine, __shfl_xor_sync(0xffffffffu, mine, d));
                const int dn = mine;                  // steps every compute warp has finished (face stores included)
                if (dn - published >= p.chunk || (dn == T && published < T)) {
                    if (lane == 0) st_release_gpu(my_flag, dn);
                    published = dn;
                }
                if (published == T) break;
                if (avail_y < T || avail_z < T) {
                    const int vy = avail_y < T ? ld_relaxed_gpu(up_y) : avail_y;
                    const int vz = avail_z < T ? ld_relaxed_gpu(up_z) : avail_z;
                    if (vy != avail_y || vz != avail_z) {
                        fence_acq_rel_gpu();
                        avail_y = vy; avail_z = vz;
                        const int al = min(avail_y >= T ? BIG : avail_y - DOS_TJ, avail_z >= T ? BIG : avail_z - DOS_TK);
                        if (lane == 0) st_release_cta(&s_allowed, al);
                        spins = 0;
                    } else {
                        if (++spins > DOS_SPIN_LIMIT) atomicExch(p.abort_flag, 1);
                        if ((spins & 255) == 0 && (ld_relaxed_gpu(p.abort_flag) || *(volatile int *)&s_abort)) {
                            avail_y = avail_z = BIG;
                            if (lane == 0) st_release_cta(&s_allowed, BIG);
                        }
                        __nanosleep(DOS_POLL_NS);
                    }
                } else {
                    __nanosleep(2 * DOS_POLL_NS);
                }
            }
            gs0 += T;
        }
    } else if (is_feed) {
        if constexpr (REALLOC) setmaxnreg_dec<REG_H>();
        while (next_item()) {
            // ------- feeder warp: bulk copies of the tile-inflow faces the upwind tiles have published -------
            // step s of octant qq needs fy_in[s][A][TK] and fz_in[s][A][TJ]: two contiguous blocks per octant.
            __syncthreads();                          // S2: s_allowed in place
            if (has_y || has_z) {
                const int qq = lane & 3, which = lane >> 2;       // lanes 0..7: (octant, y / z)
                const int oid = ((quad * 4 + qq) * p.ntk + tk) * p.ntj + tj;
                const bool mine = lane < 8 && (which == 0 ? has_y : has_z);
                const float *src = which == 0 ? p.fy + (size_t)(oid - 1) * fstride_y : p.fz + (size_t)(oid - p.ntj) * fstride_z;
                const int blk = which == 0 ? A * DOS_TK : A * DOS_TJ;                  // floats per step
                float *dst0 = which == 0 ? s_finy + qq * blk : s_finz + qq * blk;
                const unsigned bytes_all = (unsigned)((has_y ? 4 * A * DOS_TK : 0) + (has_z ? 4 * A * DOS_TJ : 0)) * 4u;
                int allowed_c = -1;
#pragma unroll 1
                for (int s = 0; s < T; ++s) {
                    // the ring slot is free once every compute warp has finished step s - RFU
                    int spins = 0;
                    for (;;) {
                        int mn = lane < NCW ? ld_acquire_cta(&s_prog[lane]) : BIG;
#pragma unroll
                        for (int d = 16; d >= 1; d >>= 1) mn = min(mn, __shfl_xor_sync(0xffffffffu, mn, d));
                        if (mn >= s - RFU + 1) break;
                        if (((++spins) & 255) == 0 && *(volatile int *)&s_abort) break;
                        __nanosleep(32);
                    }
                    while (allowed_c < s) {           // wait until the upwind tiles have published step s
                        allowed_c = ld_acquire_cta(&s_allowed);
                        if (allowed_c < s) __nanosleep(DOS_POLL_NS);
                    }
                    fence_proxy_async_all();          // the acquire above orders the upwind stores before these async reads
                    uint64_t *bar = &fin_full[(fs0 + s) % RFU];
                    if (lane == 0) mbar_arrive_expect_tx(bar, bytes_all);
                    __syncwarp();
                    if (mine) bulk_g2s(dst0 + ((fs0 + s) % RFU) * 4 * blk, src + (size_t)s * blk, (unsigned)blk * 4u, bar);
                }
                fs0 += T;
            }
            gs0 += T;
        }
    } else if (is_m2d) {
        if constexpr (REALLOC) setmaxnreg_dec<REG_H>();
        while (next_item()) {
            // ------- M2D issuer: D_q[slot] = A_lo B_hi + A_hi B_lo + A_hi B_hi -------
            __syncthreads();                          // S2
            const bool leader = elect_one();
            const unsigned idesc = umma_idesc_tf32(128, NAP);
            const unsigned a_slot_bytes = 2 * 16 * NCH * 128, a_half = 16 * NCH * 128, b_half = (NAP / 8) * NCH * 128;
            const uint64_t bdh = umma_smem_desc(smem_u32(s_bm), 128, NCH * 128), bdl = umma_smem_desc(smem_u32(s_bm) + b_half, 128, NCH * 128);
#pragma unroll 1
            for (int t = 0; t < T; ++t) {
                const unsigned gs = gs0 + t;
                TRACE(0);
                wait_bar(&a_full[gs % ASL], (gs / ASL) & 1, &s_abort, p.abort_flag);
                TRACE(1);
                wait_bar(&q_empty[gs % DQS], ((gs / DQS) & 1) ^ 1, &s_abort, p.abort_flag);
                TRACE(2);
                tc_fence_after();
                {
                    const unsigned on = (leader && !(DOS_UMMA_ABL & 4)) ? 1u : 0u;
                    const unsigned a0 = smem_u32(s_a) + (gs % ASL) * a_slot_bytes;
                    const uint64_t adh = umma_smem_desc(a0, 128, NCH * 128), adl = umma_smem_desc(a0 + a_half, 128, NCH * 128);
                    const unsigned d = tm_dq + (gs % DQS) * NAP;
                    const int nk = KP / 8;
                    for (int ks = 0; ks < nk; ++ks) umma_ss_if(on, d, adl + (uint64_t)(ks * 16), bdh + (uint64_t)(ks * 16), idesc, ks ? 1u : 0u);
                    for (int ks = 0; ks < nk; ++ks) umma_ss_if(on, d, adh + (uint64_t)(ks * 16), bdl + (uint64_t)(ks * 16), idesc, 1u);
                    for (int ks = 0; ks < nk; ++ks) umma_ss_if(on, d, adh + (uint64_t)(ks * 16), bdh + (uint64_t)(ks * 16), idesc, 1u);
                    umma_commit_if(leader ? 1u : 0u, &q_full[gs % DQS]);
                    umma_commit_if(leader ? 1u : 0u, &a_empty[gs % ASL]);
                }
                __syncwarp();
                TRACE(3);
            }
            gs0 += T;
        }
    } else if (is_d2m) {
        if constexpr (REALLOC) setmaxnreg_dec<REG_H>();
        while (next_item()) {
            // ------- D2M issuer: D_phi[slot] = psi_lo B_hi + psi_hi B_lo + psi_hi B_hi (A operand in TMEM) -------
            __syncthreads();                          // S2
            const bool leader = elect_one();
            const unsigned idesc = umma_idesc_tf32(128, NMP);
            const unsigned b_half = (NMP / 8) * (A8 / 4) * 128;
            const uint64_t bdh = umma_smem_desc(smem_u32(s_bd), 128, (A8 / 4) * 128), bdl = umma_smem_desc(smem_u32(s_bd) + b_half, 128, (A8 / 4) * 128);
#pragma unroll 1
            for (int t = 0; t < T; ++t) {
                const unsigned gs = gs0 + t;
                TRACE(0);
                wait_bar(&psi_full[gs % PSL], (gs / PSL) & 1, &s_abort, p.abort_flag);
                TRACE(1);
                wait_bar(&phi_empty[gs % DPS], ((gs / DPS) & 1) ^ 1, &s_abort, p.abort_flag);
                TRACE(2);
                tc_fence_after();
                {
                    const unsigned on = (leader && !(DOS_UMMA_ABL & 4)) ? 1u : 0u;
                    const unsigned ah = tm_psi + (gs % PSL) * 2 * A8, al = ah + A8;
                    const unsigned d = tm_dphi + (gs % DPS) * NMP;
                    const int nk = A8 / 8;
                    for (int ks = 0; ks < nk; ++ks) umma_ts_if(on, d, al + ks * 8, bdh + (uint64_t)(ks * 16), idesc, ks ? 1u : 0u);
                    for (int ks = 0; ks < nk; ++ks) umma_ts_if(on, d, ah + ks * 8, bdl + (uint64_t)(ks * 16), idesc, 1u);
                    for (int ks = 0; ks < nk; ++ks) umma_ts_if(on, d, ah + ks * 8, bdh + (uint64_t)(ks * 16), idesc, 1u);
                    umma_commit_if(leader ? 1u : 0u, &phi_full[gs % DPS]);
                    umma_commit_if(leader ? 1u : 0u, &psi_empty[gs % PSL]);
                }
                __syncwarp();
                TRACE(3);
            }
            gs0 += T;
        }
    } else if (is_split) {
        if constexpr (REALLOC) setmaxnreg_dec<REG_H>();
        while (next_item()) {
            // this warp owns octant o = 4 quad + q; the lane owns one (j,k) column of its tile
            const int o = quad * 4 + q;
            const Geom g = make_geom(p, o, tj, tk, lane);
            const int row = q * 32 + lane;
            // ------- split warp: bulk copy of each row's MP source moments, mirror signs, TF32 hi / lo, UMMA layout -------
            __syncthreads();                          // S2
            const float *qsrc = p.Q + g.cbase * MP;
            const long long qinc = (long long)g.istep * MP;
            const unsigned *sgn = s_sign + o * MP;
            const int nq = MP / 4;
            auto issue = [&](int s) {
                // one 16-byte cp.async per 4 moments of this lane's row; the lane's arrival on the ring slot's mbarrier
                // fires when they have landed
                const bool on = (unsigned)(s - g.t_lo) < (unsigned)nx;
                uint64_t *bar = &raw_full[((gs0 + s) % RAW) * 4 + q];
                if (on && !(DOS_UMMA_ABL & 1)) {
                    float *dst = s_raw + ((size_t)((gs0 + s) % RAW) * 128 + row) * MP;
                    const float *src = qsrc + qinc * s;
                    switch (nq) {
                        case 1: split_issue<1>(dst, src); break;
                        case 3: split_issue<3>(dst, src); break;
                        case 4: split_issue<4>(dst, src); break;
                        case 7: split_issue<7>(dst, src); break;
                        default: split_issue<9>(dst, src); break;
                    }
                }
                cp_async_mbar_arrive(bar);
            };
            for (int s = 0; s < LA && s < T; ++s) issue(s);
#pragma unroll 1
            for (int t = 0; t < T; ++t) {
                const unsigned gs = gs0 + t;
                TRACE(0);
                if (t + LA < T) issue(t + LA);
                TRACE(1);
                wait_bar(&raw_full[(gs % RAW) * 4 + q], (gs / RAW) & 1, &s_abort, p.abort_flag);
                TRACE(2);
                wait_bar(&a_empty[gs % ASL], ((gs / ASL) & 1) ^ 1, &s_abort, p.abort_flag);
                TRACE(3);
                const bool on = (unsigned)(t - g.t_lo) < (unsigned)nx;
                const float4 *src = reinterpret_cast<const float4 *>(s_raw + ((size_t)(gs % RAW) * 128 + row) * MP);
                // element (row, chunk c): ((row / 8) * NCH + c) * 32 + (row % 8) * 4 floats
                float4 *dh = reinterpret_cast<float4 *>(s_a + (size_t)(gs % ASL) * (2 * 16 * NCH * 32) + ((row >> 3) * NCH) * 32 + (row & 7) * 4);
                float4 *dl = dh + 16 * NCH * 8;
                switch (nq) {
                    case 1: split_row<1>(src, sgn, dh, dl, on); break;
                    case 3: split_row<3>(src, sgn, dh, dl, on); break;
                    case 4: split_row<4>(src, sgn, dh, dl, on); break;
                    case 7: split_row<7>(src, sgn, dh, dl, on); break;
                    default: split_row<9>(src, sgn, dh, dl, on); break;
                }
                fence_proxy_async_smem();             // the stores above -> the UMMA's operand reads; the row reads -> the next bulk copy
                __syncwarp();
                if (lane == 0) mbar_arrive(&a_full[gs % ASL]);
                TRACE(4);
            }
            gs0 += T;
        }
    } else if (is_epi) {
        if constexpr (REALLOC) setmaxnreg_dec<REG_H>();
        while (next_item()) {
            const int o = quad * 4 + q;
            const Geom g = make_geom(p, o, tj, tk, lane);
            // ------- epilogue warp: D_phi row -> mirror signs -> red.global.add into phi[cell][MP] -------
            __syncthreads();                          // S2
            float *phi_p = p.phi + g.cbase * MP;
            const long long pinc = (long long)g.istep * MP;
            const unsigned *sgn = s_sign + o * MP;
#pragma unroll 1
            for (int t = 0; t < T; ++t) {
                const unsigned gs = gs0 + t;
                TRACE(0);
                wait_bar(&phi_full[gs % DPS], (gs / DPS) & 1, &s_abort, p.abort_flag);
                TRACE(1);
                tc_fence_after();
                const bool on = (unsigned)(t - g.t_lo) < (unsigned)nx;
                const unsigned ta = tm_dphi + lane_base + (gs % DPS) * NMP;
                switch (MP) {
                    case 4: epilogue_row<4, 0>(ta, sgn, phi_p, on); break;
                    case 12: epilogue_row<12, 0>(ta, sgn, phi_p, on); break;
                    case 16: epilogue_row<16, 0>(ta, sgn, phi_p, on); break;
                    case 28: epilogue_row<28, 0>(ta, sgn, phi_p, on); break;
                    default: epilogue_row<36, 0>(ta, sgn, phi_p, on); break;
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&phi_empty[gs % DPS]);
                TRACE(2);
                phi_p += pinc;
            }
            gs0 += T;
        }
    } else {
        // ---------------- compute warps: diamond difference, face hand-off ----------------
        if constexpr (REALLOC) setmaxnreg_inc<REG_C>();
        while (next_item()) {
            const int o = quad * 4 + q;
            const Geom g = make_geom(p, o, tj, tk, lane);
            const int grp = warp >> 2, a0 = grp * AG;
            const int jj = lane & (DOS_TJ - 1), kk = lane / DOS_TJ;
            const bool in_y = jj == 0, in_z = kk == 0;
            const bool store_y = g.valid && jj == DOS_TJ - 1 && tj < p.ntj - 1;
            const bool store_z = g.valid && kk == DOS_TK - 1 && tk < p.ntk - 1;
            const int oid = (o * p.ntk + tk) * p.ntj + tj;
            float *fy_st = p.fy + (size_t)oid * fstride_y + kk + ((long long)(1 - DOS_TJ) * A + a0) * DOS_TK;
            float *fz_st = p.fz + (size_t)oid * fstride_z + jj + ((long long)(1 - DOS_TK) * A + a0) * DOS_TJ;
            const int fy_inc = A * DOS_TK, fz_inc = A * DOS_TJ;
            const float *finy = s_finy + (q * A + a0) * DOS_TK + kk, *finz = s_finz + (q * A + a0) * DOS_TJ + jj;
            const uint8_t *mat_p = p.mat + g.cbase;
            const int istep = g.istep, t_lo = g.t_lo;
            __syncthreads();                          // S2
            const float4 *cdd4 = reinterpret_cast<const float4 *>(s_cdd) + a0;     // (cx, cy, cz, cx+cy+cz) per angle: warp-uniform reads
            float px[AG], oy[AG], oz[AG];
#pragma unroll
            for (int r = 0; r < AG; ++r) px[r] = oy[r] = oz[r] = 0.f;
            auto mat_of = [&](int s) -> int { return ((unsigned)(s - t_lo) < (unsigned)nx) ? min((int)__ldg(mat_p + (long long)istep * s), p.n_mat - 1) : 0; };
            int m_cur = mat_of(0), m_nxt = mat_of(1);

#pragma unroll 1
            for (int t = 0; t < T; ++t) {
                const unsigned gs = gs0 + t;
                const bool act = (unsigned)(t - t_lo) < (unsigned)nx;
                const int m0 = m_cur;
                m_cur = m_nxt;
                m_nxt = mat_of(t + 2);
                TRACE(0);
                wait_bar(&q_full[gs % DQS], (gs / DQS) & 1, &s_abort, p.abort_flag, 32);
                TRACE(1);
                tc_fence_after();
                const unsigned fs = fs0 + t;
                if (has_y || has_z) wait_bar(&fin_full[fs % RFU], (fs / RFU) & 1, &s_abort, p.abort_flag, 32);
                TRACE(3);
                const int fslot = (int)(fs % RFU) * 4 * A;
                const float *rden = s_rden + m0 * A + a0;
                const float sig0 = s_sig[m0];
                const bool first_x = t == t_lo;
                const unsigned tq = tm_dq + lane_base + (gs % DQS) * NAP + a0;            // D_q columns of this warp's angles
                const unsigned tp = tm_psi + lane_base + (gs % PSL) * 2 * A8 + a0;        // psi operand columns (hi; lo at + A8)
                // The AG angles go in chunks of CH. Inside a chunk everything is straight-line code (selects, no branches),
                // so the CH independent dependency chains interleave; the set-to-zero fixup runs for the whole chunk in
                // lock-step while any lane of the warp still has a negative outflow. R12: the pinned set only grows. A
                // pinned face has outflow exactly 0, so "pinned" is read off the outflow itself (o <= 0): a face whose
                // unpinned outflow is exactly 0 may be treated as pinned, because pinning any other face lowers psi_c and
                // would pin it in the next pass anyway. A pass with nothing new to pin reproduces its input.
                // Each chunk reads its CH columns of the discrete source from tensor memory and writes its psi_c (TF32
                // hi + lo) back as the D2M's A operand, so no per-angle array outlives a chunk except the 3 face fluxes.
                constexpr int CH = (AG % 4 == 0 || AG == 7) ? 4 : (AG >= 3 ? 3 : AG);
                auto chunk = [&]<int C0>() {
                    constexpr int N = AG - C0 < CH ? AG - C0 : CH;
                    float qd[N], ix[N], yi[N], zi[N], ox[N], oyr[N], ozr[N], pc[N];
                    tmem_ld_n<N>(tq + C0, qd);
                    tmem_wait_ld();
                    bool any = false;
#pragma unroll
                    for (int e = 0; e < N; ++e) {
                        const int r = C0 + e;
                        float yin = __shfl_up_sync(0xffffffffu, oy[r], 1);
                        float zin = __shfl_up_sync(0xffffffffu, oz[r], DOS_TJ);
                        if (in_y) yin = has_y ? finy[fslot * DOS_TK + r * DOS_TK] : 0.f;        // tile inflow or vacuum
                        if (in_z) zin = has_z ? finz[fslot * DOS_TJ + r * DOS_TJ] : 0.f;
                        const float4 cc = cdd4[r];
                        ix[e] = first_x ? 0.f : px[r];
                        yi[e] = yin; zi[e] = zin;
                        const float num = fmaf(cc.x, ix[e], fmaf(cc.y, yin, fmaf(cc.z, zin, qd[e])));
                        const float c = (DOS_UMMA_ABL & 8) ? 0.f : num * rden[r];
                        pc[e] = c;
                        ox[e] = 2.f * c - ix[e]; oyr[e] = 2.f * c - yin; ozr[e] = 2.f * c - zin;
                        any |= act && fminf(ox[e], fminf(oyr[e], ozr[e])) < 0.f;
                    }
                    while (__any_sync(0xffffffffu, any)) {
                        any = false;
#pragma unroll
                        for (int e = 0; e < N; ++e) {
                            const float4 cc = cdd4[C0 + e];
                            const float gx = ox[e] > 0.f ? 1.f : 0.f, gy = oyr[e] > 0.f ? 1.f : 0.f, gz = ozr[e] > 0.f ? 1.f : 0.f;
                            const float hx = cc.x * ix[e], hy = cc.y * yi[e], hz = cc.z * zi[e];
                            const float num = fmaf(fmaf(0.5f, gx, 0.5f), hx, fmaf(fmaf(0.5f, gy, 0.5f), hy, fmaf(fmaf(0.5f, gz, 0.5f), hz, qd[e])));
                            const float den = fmaf(gx, cc.x, fmaf(gy, cc.y, fmaf(gz, cc.z, sig0)));
                            const float c = __fdividef(num, den);
                            pc[e] = c;
                            ox[e] = gx * (2.f * c - ix[e]);
                            oyr[e] = gy * (2.f * c - yi[e]);
                            ozr[e] = gz * (2.f * c - zi[e]);
                            any |= act && fminf(ox[e], fminf(oyr[e], ozr[e])) < 0.f;
                        }
                    }
                    float hi[N], lo[N];
#pragma unroll
                    for (int e = 0; e < N; ++e) {
                        const int r = C0 + e;
                        if (act) {
                            px[r] = ox[e]; oy[r] = oyr[e]; oz[r] = ozr[e];
                            if (store_y) __stcg(fy_st + r * DOS_TK, oyr[e]);
                            if (store_z) __stcg(fz_st + r * DOS_TJ, ozr[e]);
                        }
                        tf32_split(act ? pc[e] : 0.f, hi[e], lo[e]);
                    }
                    if constexpr (C0 == 0) {
                        TRACE(4);
                        wait_bar(&psi_empty[gs % PSL], ((gs / PSL) & 1) ^ 1, &s_abort, p.abort_flag, 32);
                        tc_fence_after();
                        TRACE(5);
                    }
                    tmem_st_n<N>(tp + C0, hi);
                    tmem_st_n<N>(tp + A8 + C0, lo);
                };
                [&]<int... I>(std::integer_sequence<int, I...>) { (chunk.template operator()<I * CH>(), ...); }(
                    std::make_integer_sequence<int, (AG + CH - 1) / CH>{});
                fy_st += fy_inc; fz_st += fz_inc;
                tmem_wait_st();
                tc_fence_before();
                __syncwarp();                         // also orders every lane's face stores before the progress word
                if (lane == 0) {
                    mbar_arrive(&q_empty[gs % DQS]);
                    mbar_arrive(&psi_full[gs % PSL]);
                    st_release_cta(&s_prog[warp], t + 1);
                }
                TRACE(6);
            }
            gs0 += T;
            if (has_y || has_z) fs0 += T;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc_512(tm);
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
typedef void (*sweep_u_fn)(const SweepUArgs);

struct UShape { int ag, ng; sweep_u_fn fn; };

static const UShape *umma_shape(int per_oct)
{
    // (angles per compute warp, compute warps per octant) for the level-symmetric sets: S2 1, S4 3, S6 6, S8 10,
    // S10 15, S12 21, S14 28, S16 36 angles per octant
    static const UShape shapes[] = {
        {1, 1, sweep_umma_kernel<1, 1>}, {3, 1, sweep_umma_kernel<3, 1>}, {6, 1, sweep_umma_kernel<6, 1>},
        {5, 2, sweep_umma_kernel<5, 2>}, {5, 3, sweep_umma_kernel<5, 3>}, {7, 3, sweep_umma_kernel<7, 3>},
        {7, 4, sweep_umma_kernel<7, 4>}, {12, 3, sweep_umma_kernel<12, 3>},
    };
    for (const UShape &s : shapes)
        if (s.ag * s.ng == per_oct) return &s;
    return nullptr;
}

int dos_sweep_umma_supported(int per_oct, int L)
{
    const int MP = dos_mpad(L);
    return umma_shape(per_oct) != nullptr && per_oct <= 48 && (MP == 4 || MP == 12 || MP == 16 || MP == 28 || MP == 36);
}

static size_t umma_smem(int MP, int A, int n_mat)
{
    const int KP = (MP + 7) & ~7, NCH = KP / 4, A8 = (A + 7) & ~7, NAP = (A + 15) & ~15, NMP = (MP + 15) & ~15;
    auto up = [](size_t b) { return (b + 127) & ~(size_t)127; };
    return up((size_t)RAW * 128 * MP * 4) + up((size_t)ASL * 2 * 16 * NCH * 128) + up((size_t)2 * (NAP / 8) * NCH * 128) +
           up((size_t)2 * (NMP / 8) * (A8 / 4) * 128) + up((size_t)RFU * 4 * A * DOS_TK * 4) + up((size_t)RFU * 4 * A * DOS_TJ * 4) +
           up((size_t)A * 16) + up((size_t)n_mat * A * 4) + up((size_t)n_mat * 4) + up((size_t)8 * MP * 4) + up(64 * 8) + up(32 * 4) + 128;
}

cudaError_t dos_sweep_umma_grid(int L, int per_oct, int n_mat, int n_items, int *grid_out)
{
    const UShape *s = umma_shape(per_oct);
    if (!s) return cudaErrorInvalidValue;
    const size_t smem = umma_smem(dos_mpad(L), per_oct, n_mat);
    cudaError_t e = cudaFuncSetAttribute(s->fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    if (s->ng >= 3) {
        // the register re-allocation inside the kernel must fit the CTA's allocation at launch (else it would block)
        cudaFuncAttributes fa;
        if ((e = cudaFuncGetAttributes(&fa, s->fn)) != cudaSuccess) return e;
        const int threads = (4 * s->ng + 12) * 32;
        if (fa.numRegs * threads < (umma_reg_compute(s->ng) * 4 * s->ng + umma_reg_helper(s->ng) * 12) * 32) return cudaErrorLaunchOutOfResources;
    }
    // one CTA per SM: each allocates all 512 tensor-memory columns
    *grid_out = sms < n_items ? sms : n_items;
    return cudaSuccess;
}

cudaError_t dos_launch_sweep_umma(const SweepUArgs &a, int L, int grid, cudaStream_t st)
{
    const UShape *s = umma_shape(a.per_oct);
    if (!s) return cudaErrorInvalidValue;
    const size_t smem = umma_smem(dos_mpad(L), a.per_oct, a.n_mat);
    s->fn<<<grid, (4 * s->ng + 12) * 32, smem, st>>>(a);
    return cudaGetLastError();
}
