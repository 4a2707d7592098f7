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
//               only), split into TF32 hi + lo and written to shared memory in the UMMA K-major core-matrix layout;
//               B = (2l+1) Y_lm of octant 0's angles, pre-split on the host. 3 terms (lo*hi, hi*lo, hi*hi) x K/8
//               instructions, issued by one thread, accumulator ring in TMEM.
//   cell update compute warp (octant q, angle group g) reads its AG columns of D_q straight from TMEM (tcgen05.ld),
//               takes the y/z inflow from the neighbouring lanes by shuffle (or from the staged tile-inflow faces),
//               and writes psi_c, split into hi + lo, back to TMEM (tcgen05.st) as the A operand of
//   D2M         D_phi[row][lm] = sum_a psi[row][a] w_a Y_lm(a) (A from TMEM, B from shared memory); D_phi is read back
//               (tcgen05.ld), given the mirror signs and added to phi with red.global.add.v4.
//   one warp kind  the NG compute warps of an octant also share the staging (cp.async of their 16-byte pieces of every
//               row, LA steps ahead), the split (SA steps ahead) and the read-back of D_phi (EB steps behind): lane =
//               row in all four jobs. Measured: with separate staging / read-back warps only 12 of 24 warps carried
//               cell updates, each a long dependent chain, and the SM sat at 0.2-0.4 IPC per scheduler; with every warp
//               a compute warp there are twice as many chains in flight and half as many angles per chain.
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
constexpr int LA = 4;        // steps between issuing a row's cp.async and the cell update that uses it
constexpr int SA = 2;        // steps the TF32 split (and with it the M2D) runs ahead of the cell update
constexpr int EB = 2;        // steps the read-back of D_phi lags behind the cell update
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
#ifndef DOS_UMMA_CDDC
#define DOS_UMMA_CDDC 1
#endif
#ifndef DOS_UMMA_RCP
#define DOS_UMMA_RCP 0
#endif
#ifndef DOS_UMMA_FIX
#define DOS_UMMA_FIX 0      // fixup passes: 0 angle by angle, 1 the chunk's angles together, 2 together when two or more need one
#endif
#ifndef DOS_UMMA_FIXRCP
#define DOS_UMMA_FIXRCP 1
#endif
// pauses between polls of the helper warps: a step takes ~3 us at S16 and the issuers have thousands of cycles of slack,
// while every poll is an issue slot taken from the scheduler's three compute warps (100 / 64 ns: 6.77 ms on the 256x256x64
// test, 300 / 200 ns: 6.72)
#ifndef DOS_UMMA_HSLEEP
#define DOS_UMMA_HSLEEP 300     // ns between polls of the issuer and feeder warps
#endif
#ifndef DOS_UMMA_SSLEEP
#define DOS_UMMA_SSLEEP 200     // ... of the service warp
#endif
#ifndef DOS_UMMA_ABL
#define DOS_UMMA_ABL 0        // measurement builds only: bit 0 no source-moment copies, 1 no reds, 2 no MMAs, 3 no cell update, 4 no fixup
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
__device__ __forceinline__ void wait_more(uint64_t *bar, unsigned parity, int *s_abort, int *g_abort, unsigned sleep_ns)
{
#pragma unroll 1
    for (int outer = 0; outer < WAIT_LIMIT / 1024; ++outer) {
#pragma unroll 1
        for (int spins = 0; spins < 1024; ++spins) {      // the poll itself: sleep, try, branch
            __nanosleep(sleep_ns);
            if (mbar_try_wait(bar, parity)) return;
        }
        if (*(volatile int *)s_abort) return;
    }
    *(volatile int *)s_abort = 1;
    atomicExch(g_abort, 1);
}
__device__ __forceinline__ void wait_bar(uint64_t *bar, unsigned parity, int *s_abort, int *g_abort, unsigned sleep_ns = 64)
{
    if (mbar_try_wait(bar, parity)) return;
    wait_more(bar, parity, s_abort, g_abort, sleep_ns);
}

// hi = x rounded to TF32 (round half away from zero on the bit pattern; inputs are finite), lo = x - hi (exact in
// fp32; the tensor core reads its leading 11 bits: an error <= 2^-22 |x|)
__device__ __forceinline__ void tf32_split(float x, float &hi, float &lo)
{
    hi = __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
    lo = x - hi;
}

// Register re-allocation (setmaxnreg; warp roles come in aligned groups of 4 warps, as it requires). The launch gives
// every thread R0 = 64K / threads registers (multiple of 8); the 4 helper warps keep 40 and the 4 NG compute warps share
// what that frees. setmaxnreg re-divides the CTA's OWN allocation: asking for more than the launch total blocks for
// ever, so dos_sweep_umma_grid checks the launch's register count against these numbers before anything runs.
__host__ __device__ constexpr int umma_reg_launch(int ng) { return (65536 / ((4 * ng + 4) * 32)) / 8 * 8 > 255 ? 248 : (65536 / ((4 * ng + 4) * 32)) / 8 * 8; }
__host__ __device__ constexpr int umma_reg_helper() { return 40; }
__host__ __device__ constexpr int umma_reg_compute(int ng) { return umma_reg_launch(ng) + (umma_reg_launch(ng) - umma_reg_helper()) / ng / 8 * 8; }
#ifndef DOS_UMMA_REALLOC
#define DOS_UMMA_REALLOC 1
#endif
__host__ __device__ constexpr bool umma_realloc(int ag, int ng) { return DOS_UMMA_REALLOC && ng >= 2 && ag >= 7; }

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

// One 16-byte piece (4 moments) of a row: mirror signs, TF32 hi / lo, into the UMMA core-matrix layout.
__device__ __forceinline__ void split_piece(const float4 *src, const unsigned *sgn, float4 *dh, float4 *dl, bool on)
{
    const float4 x = on ? *src : make_float4(0.f, 0.f, 0.f, 0.f);
    const uint4 s4 = *reinterpret_cast<const uint4 *>(sgn);
    float4 h, l;
    tf32_split(__uint_as_float(__float_as_uint(x.x) ^ s4.x), h.x, l.x);
    tf32_split(__uint_as_float(__float_as_uint(x.y) ^ s4.y), h.y, l.y);
    tf32_split(__uint_as_float(__float_as_uint(x.z) ^ s4.z), h.z, l.z);
    tf32_split(__uint_as_float(__float_as_uint(x.w) ^ s4.w), h.w, l.w);
    *dh = h;
    *dl = l;
}

// Warp roles (NG compute warps per octant, AG angles each):
//   [0, 4 NG)   compute: octant q = warp % 4, angle group g = warp / 4 (also: its share of staging, split, read-back)
//   4 NG        M2D issuer (one elected lane)      4 NG + 1   D2M issuer
//   4 NG + 2    feeder (tile-inflow faces)         4 NG + 3   service (global hand-off flags)
// REFL: the variant with reflective mesh faces (lagged boundary buffers); the vacuum-only variant carries none of it.
template <int AG, int NG, bool REFL>
__global__ void __launch_bounds__((4 * NG + 4) * 32, 1) sweep_umma_kernel(const SweepUArgs p)
{
    const int refl = REFL ? p.refl : 0;
    size_t sh = 0;           // byte offset of the item's problem of the position batch: Q, phi, faces, boundaries, done
    auto mv = [&sh](auto *ptr) { return reinterpret_cast<decltype(ptr)>(reinterpret_cast<size_t>(ptr) + sh); };
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int A = AG * NG, A8 = (A + 7) & ~7, NAP = (A + 15) & ~15;      // the host picks the instance with AG * NG = per_oct
    const int MP = p.MP, KP = (MP + 7) & ~7, NCH = KP / 4, NMP = (MP + 15) & ~15;
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
    float *s_zero = reinterpret_cast<float *>(carve((size_t)A * DOS_TJ * 4));                   // vacuum inflow: [A][TJ] zeros
    uint64_t *bars = reinterpret_cast<uint64_t *>(carve(64 * 8));
    int *s_prog = reinterpret_cast<int *>(carve(32 * 4));                                       // [NCW] steps finished per compute warp
    uint64_t *raw_full = bars;            // [RAW][4 octants]
    uint64_t *a_full = bars + 16;         // [ASL]
    uint64_t *q_full = bars + 20;         // [DQS]
    uint64_t *q_empty = bars + 24;
    uint64_t *psi_full = bars + 28;       // [PSL]
    uint64_t *phi_full = bars + 32;       // [DPS]
    uint64_t *phi_empty = bars + 34;
    uint64_t *fin_full = bars + 36;       // [RFU]
    __shared__ int s_item, s_allowed, s_abort;
    __shared__ unsigned s_tmem;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, q = warp & 3;
    const bool is_m2d = warp == NCW, is_d2m = warp == NCW + 1, is_feed = warp == NCW + 2, is_service = warp == NCW + 3;
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
    for (int i = tid; i < A * DOS_TJ; i += blockDim.x) s_zero[i] = 0.f;
    if (tid == 0) {
        for (int i = 0; i < 16; ++i) mbar_init(&raw_full[i], 32 * NG);      // one cp.async arrival per thread of the octant's warps
        for (int i = 0; i < ASL; ++i) mbar_init(&a_full[i], NCW);
        for (int i = 0; i < DQS; ++i) { mbar_init(&q_full[i], 1); mbar_init(&q_empty[i], NCW); }
        for (int i = 0; i < PSL; ++i) mbar_init(&psi_full[i], NCW);
        for (int i = 0; i < DPS; ++i) { mbar_init(&phi_full[i], 1); mbar_init(&phi_empty[i], NCW); }
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
    if (warp < 4) {
        // the K padding columns of the psi operands must be finite (they meet zero rows of B): zero them once
        float z[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        for (int c = 0; c < PSL * 2 * A8; c += 8) tmem_st<8>(tm_psi + lane_base + c, z);
        tmem_wait_st();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    unsigned gs0 = 0;      // global step counter at the start of the current item (ring slots and phases follow it)
    unsigned fs0 = 0;      // the same for the tile-inflow ring, which only items with an upwind tile use
    int quad = 0, tj = 0, tk = 0, fid = 0;
    bool has_y = false, has_z = false;
#if DOS_UMMA_TRACE
    bool trace_on = false;
    long long *trace_buf = reinterpret_cast<long long *>(p.fz);      // measurement build: the z-face buffer of item 0 is sacrificed
#endif
    // every role runs its own loop over the work items; all of them meet in the two barriers of next_item()
    auto next_item = [&]() -> bool {
        __syncthreads();                              // every role has drained the previous item
        if (tid == 0) s_item = atomicAdd(p.queue, 1);
        if (tid < NCW) s_prog[tid] = 0;
        __syncthreads();
        if (s_item >= p.n_items) return false;
        const int item = s_item / p.n_batch;
        sh = (size_t)(s_item - item * p.n_batch) * p.slot_stride;
        const int packed = p.items[item];
        quad = packed & 7; tj = (packed >> 3) & 0x3FFF; tk = packed >> 17;
        fid = (quad * p.ntk + tk) * p.ntj + tj;      // hand-off flag of this (quad, tile)
        has_y = tj > 0 || (refl & 2); has_z = tk > 0 || (refl & 4);      // there is y / z inflow to stage (else vacuum)
#if DOS_UMMA_TRACE
        trace_on = s_item == 601;
#endif
        return true;
    };

    constexpr bool REALLOC = umma_realloc(AG, NG);
    if (is_service) {
        if constexpr (REALLOC) setmaxnreg_dec<umma_reg_helper()>();
        while (next_item()) {
            // ------- service warp: publishes this item's progress, follows the two upwind items' progress -------
            const bool up_tile_y = tj > 0, up_tile_z = tk > 0;       // boundary inflow (reflective) needs no hand-off
            int *done = mv(p.done);
            const int *up_y = done + (up_tile_y ? fid - 1 : fid), *up_z = done + (up_tile_z ? fid - p.ntj : fid);
            int *my_flag = done + fid;
            int avail_y = up_tile_y ? 0 : BIG, avail_z = up_tile_z ? 0 : BIG;
            if (lane == 0) s_allowed = (up_tile_y || up_tile_z) ? -1 : BIG;
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
                        __nanosleep(DOS_UMMA_SSLEEP);
                    }
                } else {
                    __nanosleep(4 * DOS_UMMA_SSLEEP);
                }
            }
            gs0 += T;
        }
    } else if (is_feed) {
        if constexpr (REALLOC) setmaxnreg_dec<umma_reg_helper()>();
        while (next_item()) {
            // ------- feeder warp: bulk copies of the tile-inflow faces the upwind tiles have published -------
            // step s of octant qq needs fy_in[s][A][TK] and fz_in[s][A][TJ]: two contiguous blocks per octant.
            __syncthreads();                          // S2: s_allowed in place
            if (has_y || has_z) {
                const int qq = lane & 3, which = lane >> 2;       // lanes 0..7: (octant, y / z)
                const int oo = quad * 4 + qq;
                const int oid = (oo * p.ntk + tk) * p.ntj + tj;
                const bool mine = lane < 8 && (which == 0 ? has_y : has_z);
                // upwind tile's face buffer -- or, on a reflective mesh boundary, what the mirror octant's last tile
                // wrote there in the previous sweep (same layout: the boundary is a virtual upwind tile)
                const float *src = mv(which == 0 ? (tj > 0 ? p.fy + (size_t)(oid - 1) * fstride_y : p.by_in + (size_t)((oo ^ 2) * p.ntk + tk) * fstride_y)
                                                 : (tk > 0 ? p.fz + (size_t)(oid - p.ntj) * fstride_z : p.bz_in + (size_t)((oo ^ 4) * p.ntj + tj) * fstride_z));
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
                        __nanosleep(DOS_UMMA_HSLEEP);
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
        if constexpr (REALLOC) setmaxnreg_dec<umma_reg_helper()>();
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
                wait_bar(&a_full[gs % ASL], (gs / ASL) & 1, &s_abort, p.abort_flag, DOS_UMMA_HSLEEP);
                TRACE(1);
                wait_bar(&q_empty[gs % DQS], ((gs / DQS) & 1) ^ 1, &s_abort, p.abort_flag, DOS_UMMA_HSLEEP);
                TRACE(2);
                tc_fence_after();
                {
                    const unsigned on = (leader && !(DOS_UMMA_ABL & 4)) ? 1u : 0u;
                    const unsigned a0 = smem_u32(s_a) + (gs % ASL) * a_slot_bytes;
                    const uint64_t adh = umma_smem_desc(a0, 128, NCH * 128), adl = umma_smem_desc(a0 + a_half, 128, NCH * 128);
                    const unsigned d = tm_dq + (gs % DQS) * NAP;
                    // K / 8 instructions per term, unrolled for the K of P0, P2-P3, P4-P5 (the issue is a serial chain
                    // in one thread: every instruction saved shortens the path split -> M2D -> cell update)
                    auto issue = [&]<int NK>() {
#pragma unroll
                        for (int ks = 0; ks < NK; ++ks) umma_ss_if(on, d, adl + (uint64_t)(ks * 16), bdh + (uint64_t)(ks * 16), idesc, ks ? 1u : 0u);
#pragma unroll
                        for (int ks = 0; ks < NK; ++ks) umma_ss_if(on, d, adh + (uint64_t)(ks * 16), bdl + (uint64_t)(ks * 16), idesc, 1u);
#pragma unroll
                        for (int ks = 0; ks < NK; ++ks) umma_ss_if(on, d, adh + (uint64_t)(ks * 16), bdh + (uint64_t)(ks * 16), idesc, 1u);
                    };
                    switch (KP / 8) {
                    case 1: issue.template operator()<1>(); break;
                    case 2: issue.template operator()<2>(); break;
                    case 4: issue.template operator()<4>(); break;
                    default: issue.template operator()<5>(); break;
                    }
                    // the accumulator is ready, and with it the A slot is free again (one commit tells both)
                    umma_commit_if(leader ? 1u : 0u, &q_full[gs % DQS]);
                }
                __syncwarp();
                TRACE(3);
            }
            gs0 += T;
        }
    } else if (is_d2m) {
        if constexpr (REALLOC) setmaxnreg_dec<umma_reg_helper()>();
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
                wait_bar(&psi_full[gs % PSL], (gs / PSL) & 1, &s_abort, p.abort_flag, DOS_UMMA_HSLEEP);
                TRACE(1);
                wait_bar(&phi_empty[gs % DPS], ((gs / DPS) & 1) ^ 1, &s_abort, p.abort_flag, DOS_UMMA_HSLEEP);
                TRACE(2);
                tc_fence_after();
                {
                    const unsigned on = (leader && !(DOS_UMMA_ABL & 4)) ? 1u : 0u;
                    const unsigned ah = tm_psi + (gs % PSL) * 2 * A8, al = ah + A8;
                    const unsigned d = tm_dphi + (gs % DPS) * NMP;
                    constexpr int nk = A8 / 8;
#pragma unroll
                    for (int ks = 0; ks < nk; ++ks) umma_ts_if(on, d, al + ks * 8, bdh + (uint64_t)(ks * 16), idesc, ks ? 1u : 0u);
#pragma unroll
                    for (int ks = 0; ks < nk; ++ks) umma_ts_if(on, d, ah + ks * 8, bdl + (uint64_t)(ks * 16), idesc, 1u);
#pragma unroll
                    for (int ks = 0; ks < nk; ++ks) umma_ts_if(on, d, ah + ks * 8, bdh + (uint64_t)(ks * 16), idesc, 1u);
                    // D_phi is ready, and with it the psi operand slot is free again
                    umma_commit_if(leader ? 1u : 0u, &phi_full[gs % DPS]);
                }
                __syncwarp();
                TRACE(3);
            }
            gs0 += T;
        }
    } else {
        // ---------------- compute warps ----------------
        if constexpr (REALLOC) setmaxnreg_inc<umma_reg_compute(NG)>();
        while (next_item()) {
            const int o = quad * 4 + q;               // this warp's octant; the lane owns one (j,k) column of its tile
            const Geom g = make_geom(p, o, tj, tk, lane);
            const int row = q * 32 + lane;
            const int grp = warp >> 2, a0 = grp * AG;
            const int jj = lane & (DOS_TJ - 1), kk = lane / DOS_TJ;
            const bool in_y = jj == 0, in_z = kk == 0;
            // the tile's last j / k lanes hand their outflow to the downwind tile; on the mesh's last tile row (ragged:
            // lane (ny - 1) % 8 / (nz - 1) % 4) to the reflective boundary buffer, or nowhere (vacuum)
            const bool last_tj = tj == p.ntj - 1, last_tk = tk == p.ntk - 1;
            const int jst = last_tj ? (p.ny - 1) % DOS_TJ : DOS_TJ - 1, kst = last_tk ? (p.nz - 1) % DOS_TK : DOS_TK - 1;
            const bool store_y = g.valid && jj == jst && (!last_tj || (refl & 2));
            const bool store_z = g.valid && kk == kst && (!last_tk || (refl & 4));
            const int oid = (o * p.ntk + tk) * p.ntj + tj;
            float *fy_st = mv((REFL && last_tj) ? p.by_out + (size_t)(o * p.ntk + tk) * fstride_y : p.fy + (size_t)oid * fstride_y) + kk +
                           ((long long)(-jst) * A + a0) * DOS_TK;
            float *fz_st = mv((REFL && last_tk) ? p.bz_out + (size_t)(o * p.ntj + tj) * fstride_z : p.fz + (size_t)oid * fstride_z) + jj +
                           ((long long)(-kst) * A + a0) * DOS_TJ;
            const int fy_inc = A * DOS_TK, fz_inc = A * DOS_TJ;
            const float *finy0 = s_finy + (q * A + a0) * DOS_TK + kk, *finz0 = s_finz + (q * A + a0) * DOS_TJ + jj;
            const int istep = g.istep, t_lo = g.t_lo;
            const unsigned *sgn = s_sign + o * MP;
            const int nq = MP / 4;                                       // 16-byte pieces of a row
            // Global traffic is laid out piece-major, not row-major: the octant's 32 rows of a step are 32 nq pieces of
            // 16 bytes; lane l of the octant's warp grp moves pieces (k NG + grp) 32 + l. Consecutive lanes then touch
            // consecutive 16 bytes of the same row (2-3 lines per row) where "lane = row" costs one L1 wavefront per
            // lane and piece: measured, those wavefronts (~2 cycles each, ~3000 per step) were the sweep's bound.
            // Per piece: its 16-byte offset in Q / phi at step 0 and (piece index in the row) << 16 | (row's first step).
            constexpr int KPL = (9 + NG - 1) / NG;
            int poff[KPL];
            unsigned pmeta[KPL];
#pragma unroll
            for (int k = 0; k < KPL; ++k) {
                const int i = (k * NG + grp) * 32 + lane, r = i / nq, c = i - r * nq;
                const Geom gr = make_geom(p, o, tj, tk, r & 31);
                const bool ok = i < 32 * nq && gr.valid;
                poff[k] = ok ? (int)((gr.cbase * MP + 4 * c) >> 2) : 0;
                pmeta[k] = ok ? ((unsigned)c << 16) | (unsigned)gr.t_lo : 0x7fffu;
            }
            const int cstep16 = istep * nq;                              // 16-byte units between a column's consecutive cells
            const float *Qb = mv(p.Q);
            float *phib = mv(p.phi);
            // material ids: the column's cells are consecutive bytes, so one aligned 32-bit load serves 4 steps
            const int jp_ = tj * DOS_TJ + jj, kp_ = tk * DOS_TK + kk;
            const int jg = (o & 2) ? p.ny - 1 - jp_ : jp_, kg = (o & 4) ? p.nz - 1 - kp_ : kp_;
            const uint8_t *mat_col = p.mat + (g.valid ? ((size_t)kg * p.ny + jg) * nx : 0);
            const bool mat4 = (nx & 3) == 0;
            __syncthreads();                          // S2
#if !DOS_UMMA_CDDC
            const float4 *cdd4 = reinterpret_cast<const float4 *>(s_cdd) + a0;     // (cx, cy, cz, cx+cy+cz) per angle: warp-uniform reads
#endif

            // staging: this lane's pieces of its row of step s, by cp.async; the thread's arrival on the ring slot's
            // mbarrier fires when they have landed
            auto stage = [&](int s) {
                const unsigned gsx = gs0 + s;
                float *dst = s_raw + ((size_t)(gsx % RAW) * 128 + q * 32) * MP + 4 * (grp * 32 + lane);
#pragma unroll
                for (int k = 0; k < KPL; ++k)
                    if ((unsigned)(s - (int)(pmeta[k] & 0xffffu)) < (unsigned)nx && !(DOS_UMMA_ABL & 1))
                        cp_async16(dst + k * (NG * 128), Qb + ((long long)poff[k] + (long long)cstep16 * s) * 4);
                cp_async_mbar_arrive(&raw_full[(gsx % RAW) * 4 + q]);
            };
            // split: this lane's pieces of its row of step s -> mirror signs, TF32 hi / lo, UMMA layout -> a_full
            // (the A slot of step s was last read by the M2D of step s - ASL: the caller has seen that one's q_full)
            auto split = [&](int s, bool landed) {
                const unsigned gsx = gs0 + s;
                if (!landed) wait_more(&raw_full[(gsx % RAW) * 4 + q], (gsx / RAW) & 1, &s_abort, p.abort_flag, 32);
                const bool on = (unsigned)(s - t_lo) < (unsigned)nx;
                const float4 *src = reinterpret_cast<const float4 *>(s_raw + ((size_t)(gsx % RAW) * 128 + row) * MP);
                // element (row, piece c): ((row / 8) * NCH + c) * 32 + (row % 8) * 4 floats
                float4 *dh = reinterpret_cast<float4 *>(s_a + (size_t)(gsx % ASL) * (2 * 16 * NCH * 32) + ((row >> 3) * NCH) * 32 + (row & 7) * 4);
                float4 *dl = dh + 16 * NCH * 8;
                for (int c = grp; c < nq; c += NG) split_piece(src + c, sgn + 4 * c, dh + c * 8, dl + c * 8, on);
                fence_proxy_async_smem();             // the stores above -> the UMMA's operand reads
                __syncwarp();
                if (lane == 0) mbar_arrive(&a_full[gsx % ASL]);
            };
            // read-back: D_phi of step s leaves tensor memory row by row (lane = row: this warp's pieces grp, grp + NG, ..),
            // is turned piece-major through shared memory, gets the mirror signs and goes into phi with red.global.add.v4.
            // The turning buffer is the staging slot the split of step s + EB + SA has just consumed: this warp writes
            // only the pieces it read there itself; the octant's warps meet in a named barrier before they read each
            // other's pieces, and that same barrier one step later orders these reads before the slot's next cp.async.
            auto readback = [&](int s, bool ready) {
                const unsigned gsx = gs0 + s;
                if (!ready) wait_more(&phi_full[gsx % DPS], (gsx / DPS) & 1, &s_abort, p.abort_flag, 32);
                tc_fence_after();
                const unsigned ta = tm_dphi + lane_base + (gsx % DPS) * NMP;
                float *rb = s_raw + ((size_t)((gsx + EB + SA) % RAW) * 128 + q * 32) * MP;
                float4 *mine = reinterpret_cast<float4 *>(rb + lane * MP);
                for (int c = grp; c < nq; c += 3 * NG) {      // three pieces in flight per tcgen05.wait::ld (warp-uniform conditions)
                    float v0[4], v1[4], v2[4];
                    tmem_ld<4>(ta + 4 * c, v0);
                    if (c + NG < nq) tmem_ld<4>(ta + 4 * (c + NG), v1);
                    if (c + 2 * NG < nq) tmem_ld<4>(ta + 4 * (c + 2 * NG), v2);
                    tmem_wait_ld();
                    mine[c] = make_float4(v0[0], v0[1], v0[2], v0[3]);
                    if (c + NG < nq) mine[c + NG] = make_float4(v1[0], v1[1], v1[2], v1[3]);
                    if (c + 2 * NG < nq) mine[c + 2 * NG] = make_float4(v2[0], v2[1], v2[2], v2[3]);
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&phi_empty[gsx % DPS]);
                if constexpr (NG > 1) asm volatile("bar.sync %0, %1;" ::"r"(1 + q), "n"(32 * NG) : "memory");
                const float4 *pm = reinterpret_cast<const float4 *>(rb) + grp * 32 + lane;
#pragma unroll
                for (int k = 0; k < KPL; ++k)
                    if ((unsigned)(s - (int)(pmeta[k] & 0xffffu)) < (unsigned)nx && !(DOS_UMMA_ABL & 2)) {
                        const float4 v = pm[k * (NG * 32)];
                        const uint4 s4 = *reinterpret_cast<const uint4 *>(sgn + 4 * (pmeta[k] >> 16));
                        red_add_v4(phib + ((long long)poff[k] + (long long)cstep16 * s) * 4, __uint_as_float(__float_as_uint(v.x) ^ s4.x),
                                   __uint_as_float(__float_as_uint(v.y) ^ s4.y), __uint_as_float(__float_as_uint(v.z) ^ s4.z),
                                   __uint_as_float(__float_as_uint(v.w) ^ s4.w));
                    }
            };

            // x faces: the column's inflow is vacuum or the mirror octant's outflow of the previous sweep
            // (reflective); px starts as that inflow and is only touched while the lane is active
            const size_t bxi = g.valid ? (size_t)kg * p.ny + jg : 0, bxs = (size_t)p.nz * p.ny;
            const bool refl_x = (refl & 1) && g.valid;
            const int t_last = g.valid ? t_lo + nx - 1 : -1;
            float px[AG], oy[AG], oz[AG];
#pragma unroll
            for (int r = 0; r < AG; ++r) px[r] = oy[r] = oz[r] = 0.f;
            // material word of the next 4 cells in travel order, fetched 3 steps before its first cell (nx % 4 != 0: bytes)
            auto mat_word = [&](int xl) -> unsigned {       // xl: first cell of the word, counted along the travel direction
                return __ldg(reinterpret_cast<const unsigned *>(mat_col + (istep > 0 ? xl : nx - 4 - xl)));
            };
            unsigned mw = 0, mw_nxt = (mat4 && g.valid) ? mat_word(0) : 0;
            for (int s = 0; s < LA && s < T; ++s) stage(s);
            for (int s = 0; s < SA && s < T; ++s) split(s, false);

#pragma unroll 1
            for (int t = 0; t < T; ++t) {
                const unsigned gs = gs0 + t;
                const bool act = (unsigned)(t - t_lo) < (unsigned)nx;
                const int xl = t - t_lo;              // the lane's cell of this step, counted along the travel direction
                int m0 = 0;
                if (mat4) {
                    if (act && (xl & 3) == 0) mw = mw_nxt;
                    if (act && (xl & 3) == 1 && xl + 3 < nx) mw_nxt = mat_word(xl + 3);
                    m0 = (int)((mw >> (8 * (istep > 0 ? (xl & 3) : 3 - (xl & 3)))) & 255u);
                } else if (act) {
                    m0 = (int)__ldg(mat_col + (istep > 0 ? xl : nx - 1 - xl));
                }
                m0 = min(m0, p.n_mat - 1);
                TRACE(0);
                // The step's four hand-offs are polled up front, together (a try_wait takes ~100 cycles to answer even
                // when the phase is long over); whatever has not arrived yet is waited for where it is needed.
                const unsigned fs = fs0 + t;
                const bool have_in = has_y || has_z, do_split = t + SA < T, do_rb = t >= EB;
                const bool r_q = mbar_try_wait(&q_full[gs % DQS], (gs / DQS) & 1);
                const bool r_f = have_in ? mbar_try_wait(&fin_full[fs % RFU], (fs / RFU) & 1) : true;
                const bool r_r = do_split ? mbar_try_wait(&raw_full[((gs + SA) % RAW) * 4 + q], ((gs + SA) / RAW) & 1) : true;
                const bool r_p = do_rb ? mbar_try_wait(&phi_full[(gs - EB) % DPS], ((gs - EB) / DPS) & 1) : true;
                if (t + LA < T) stage(t + LA);
                if (!r_q) wait_more(&q_full[gs % DQS], (gs / DQS) & 1, &s_abort, p.abort_flag, 32);
                TRACE(1);
                tc_fence_after();
                // M2D of step t is done: its A slot takes the split of step t + SA (so that M2D has a whole cell update
                // of lead); D2M of step t - EB is done once its D_phi is there: its psi slot is the one this step writes
                if (do_split) split(t + SA, r_r);
                TRACE(2);
                if (do_rb) readback(t - EB, r_p);
                TRACE(3);
                if (!r_f) wait_more(&fin_full[fs % RFU], (fs / RFU) & 1, &s_abort, p.abort_flag, 32);
                TRACE(4);
                const int fslot = (int)(fs % RFU) * 4 * A;
#if !DOS_UMMA_RCP
                const float *rden = s_rden + m0 * A + a0;
#endif
                const float sig0 = s_sig[m0];
                if (t == t_lo) {                      // the lane's first cell: seed the x face with the column's inflow
#pragma unroll
                    for (int r = 0; r < AG; ++r) {
                        px[r] = 0.f;
                        if constexpr (REFL)
                            if (refl_x) px[r] = __ldcg(mv(p.bx_in) + ((size_t)(o ^ 1) * A + a0 + r) * bxs + bxi);
                    }
                }
                const bool last_x = REFL && refl_x && t == t_last;
                const bool st_y = store_y && act, st_z = store_z && act;
                const float *finy = has_y ? finy0 + fslot * DOS_TK : s_zero, *finz = has_z ? finz0 + fslot * DOS_TJ : s_zero;
                const unsigned tq = tm_dq + lane_base + (gs % DQS) * NAP + a0;            // D_q columns of this warp's angles
                const unsigned tp = tm_psi + lane_base + (gs % PSL) * 2 * A8 + a0;        // psi operand columns (hi; lo at + A8)
                // The AG angles go in chunks of CH. Inside a chunk everything is straight-line code (selects, no branches),
                // so the CH independent dependency chains interleave; the set-to-zero fixup runs for the whole chunk in
                // lock-step while any lane of the warp still has a negative outflow. R12: the pinned set only grows. A
                // pinned face has outflow exactly 0, so "pinned" is read off the outflow itself (o <= 0): a face whose
                // unpinned outflow is exactly 0 may be treated as pinned, because pinning any other face lowers psi_c and
                // would pin it in the next pass anyway. A pass with nothing new to pin reproduces its input.
                // Each chunk reads its columns of the discrete source from tensor memory and writes its psi_c (TF32
                // hi + lo) back as the D2M's A operand, so no per-angle array outlives a chunk except the 3 face fluxes.
#ifndef DOS_UMMA_CH
#define DOS_UMMA_CH 3
#endif
                // (the reflective variant of the widest shape is short of registers: smaller chunks, no prefetch)
                constexpr bool TIGHT = REFL && AG >= 12;
                constexpr int CHW = TIGHT ? 3 : DOS_UMMA_CH;
                constexpr int CH = AG <= CHW ? AG : (AG % CHW == 0 ? CHW : (AG % 3 == 0 ? 3 : 4));
#ifndef DOS_UMMA_QPF
#define DOS_UMMA_QPF 0
#endif
                float qn[CH];                         // the next chunk's columns of D_q, in flight while this chunk computes
                if constexpr (DOS_UMMA_QPF && !TIGHT) tmem_ld_n<(AG < CH ? AG : CH)>(tq, qn);
                auto chunk = [&]<int C0>() {
                    constexpr int N = AG - C0 < CH ? AG - C0 : CH;
                    float qd[N], ix[N], yi[N], zi[N], ox[N], oyr[N], ozr[N], pc[N];
                    if constexpr (DOS_UMMA_QPF && !TIGHT) {
                        tmem_wait_ld();
#pragma unroll
                        for (int e = 0; e < N; ++e) qd[e] = qn[e];
                        if constexpr (C0 + CH < AG) tmem_ld_n<(AG - C0 - CH < CH ? AG - C0 - CH : CH)>(tq + C0 + CH, qn);
                    } else {
                        tmem_ld_n<N>(tq + C0, qd);
                        tmem_wait_ld();
                    }
                    unsigned negm = 0;                // bit e: angle e of the chunk has a negative outflow in this (active) lane
#pragma unroll
                    for (int e = 0; e < N; ++e) {
                        const int r = C0 + e;
                        // y / z inflow: the neighbouring lane's outflow of the previous step; lanes on the tile's inflow edge
                        // take the staged face instead (a zero block stands in for vacuum)
                        float yin = __shfl_up_sync(0xffffffffu, oy[r], 1);
                        float zin = __shfl_up_sync(0xffffffffu, oz[r], DOS_TJ);
                        if (in_y) yin = finy[r * DOS_TK];
                        if (in_z) zin = finz[r * DOS_TJ];
#if DOS_UMMA_CDDC
                        const float4 cc = make_float4(p.cddc[(a0 + r) * 4], p.cddc[(a0 + r) * 4 + 1], p.cddc[(a0 + r) * 4 + 2], p.cddc[(a0 + r) * 4 + 3]);
#else
                        const float4 cc = cdd4[r];
#endif
                        ix[e] = px[r];
                        yi[e] = yin; zi[e] = zin;
                        const float num = fmaf(cc.x, ix[e], fmaf(cc.y, yin, fmaf(cc.z, zin, qd[e])));
#if DOS_UMMA_RCP
                        float rd;                     // 1 / (sigma_t + cx + cy + cz): one MUFU instead of a per-lane table look-up
                        asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rd) : "f"(sig0 + cc.w));
                        const float c = (DOS_UMMA_ABL & 8) ? 0.f : num * rd;
#else
                        const float c = (DOS_UMMA_ABL & 8) ? 0.f : num * rden[r];
#endif
                        pc[e] = c;
                        ox[e] = 2.f * c - ix[e]; oyr[e] = 2.f * c - yin; ozr[e] = 2.f * c - zin;
                        if (fminf(ox[e], fminf(oyr[e], ozr[e])) < 0.f) negm |= 1u << e;
                    }
                    if (!act) negm = 0;
                    // Set-to-zero fixup with rebalance, angle by angle but only for angles some lane of the warp needs it
                    // for: all lanes run the pass in lock-step (a lane with nothing new to pin reproduces its values).
                    if (!(DOS_UMMA_ABL & 16) && __any_sync(0xffffffffu, negm != 0)) {
                        auto pass = [&](int e) -> bool {      // one fixup pass of angle e; true if the lane found a new negative outflow
#if DOS_UMMA_CDDC
                            const float4 cc = make_float4(p.cddc[(a0 + C0 + e) * 4], p.cddc[(a0 + C0 + e) * 4 + 1], p.cddc[(a0 + C0 + e) * 4 + 2], 0.f);
#else
                            const float4 cc = cdd4[C0 + e];
#endif
                            const float gx = ox[e] > 0.f ? 1.f : 0.f, gy = oyr[e] > 0.f ? 1.f : 0.f, gz = ozr[e] > 0.f ? 1.f : 0.f;
                            const float hx = cc.x * ix[e], hy = cc.y * yi[e], hz = cc.z * zi[e];
                            const float num = fmaf(fmaf(0.5f, gx, 0.5f), hx, fmaf(fmaf(0.5f, gy, 0.5f), hy, fmaf(fmaf(0.5f, gz, 0.5f), hz, qd[e])));
                            const float den = fmaf(gx, cc.x, fmaf(gy, cc.y, fmaf(gz, cc.z, sig0)));
#if DOS_UMMA_FIXRCP
                            float rd;                 // den >= sigma_t > 0 and finite: no range handling needed
                            asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rd) : "f"(den));
                            const float c = num * rd;
#else
                            const float c = __fdividef(num, den);
#endif
                            pc[e] = c;
                            ox[e] = gx * (2.f * c - ix[e]);
                            oyr[e] = gy * (2.f * c - yi[e]);
                            ozr[e] = gz * (2.f * c - zi[e]);
                            return act && fminf(ox[e], fminf(oyr[e], ozr[e])) < 0.f;
                        };
#if DOS_UMMA_FIX == 0
#pragma unroll
                        for (int e = 0; e < N; ++e) {
                            bool neg = (negm >> e) & 1u;
                            while (__any_sync(0xffffffffu, neg)) neg = pass(e);
                        }
#else
                        // angles some lane needs a pass for (warp-uniform); with two or more, the passes of all the chunk's
                        // angles run together so that their dependent chains overlap; a pass of an angle nobody needs it for
                        // reproduces its values
                        const unsigned wm = __reduce_or_sync(0xffffffffu, negm);
                        if (DOS_UMMA_FIX == 1 || (wm & (wm - 1))) {
                            bool neg = true;
                            while (__any_sync(0xffffffffu, neg)) {
                                neg = false;
#pragma unroll
                                for (int e = 0; e < N; ++e) neg |= pass(e);
                            }
                        } else {
#pragma unroll
                            for (int e = 0; e < N; ++e)
                                if (wm >> e & 1u) {
                                    bool neg = true;
                                    while (__any_sync(0xffffffffu, neg)) neg = pass(e);
                                }
                        }
#endif
                    }
                    // Lanes outside their x range compute on whatever they hold: nothing reads it (their neighbours are
                    // outside too, their rows are skipped by the read-back, their stores are predicated off, and px is
                    // re-seeded from the boundary value at the lane's first cell).
                    float hi[N], lo[N];
#pragma unroll
                    for (int e = 0; e < N; ++e) {
                        const int r = C0 + e;
                        px[r] = ox[e]; oy[r] = oyr[e]; oz[r] = ozr[e];
                        if (st_y) __stcg(fy_st + r * DOS_TK, oyr[e]);
                        if (st_z) __stcg(fz_st + r * DOS_TJ, ozr[e]);
                        if constexpr (REFL)
                            if (last_x) __stcg(mv(p.bx_out) + ((size_t)o * A + a0 + r) * bxs + bxi, ox[e]);
                        tf32_split(pc[e], hi[e], lo[e]);
                    }
                    tmem_st_n<N>(tp + C0, hi);
                    tmem_st_n<N>(tp + A8 + C0, lo);
                    if constexpr (C0 == 0) TRACE(5);
                };
                [&]<int... I>(std::integer_sequence<int, I...>) { (chunk.template operator()<I * CH>(), ...); }(
                    std::make_integer_sequence<int, (AG + CH - 1) / CH>{});
                fy_st += fy_inc; fz_st += fz_inc;
                TRACE(6);
                tmem_wait_st();
                tc_fence_before();
                __syncwarp();                         // also orders every lane's face stores before the progress word
                if (lane == 0) {
                    mbar_arrive(&q_empty[gs % DQS]);
                    mbar_arrive(&psi_full[gs % PSL]);
                    st_release_cta(&s_prog[warp], t + 1);
                }
                TRACE(7);
            }
            for (int s = T - EB > 0 ? T - EB : 0; s < T; ++s) readback(s, false);
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

struct UShape { int ag, ng; sweep_u_fn fn[2]; };      // [vacuum only, reflective faces]
#define USHAPE(AG, NG) {AG, NG, {sweep_umma_kernel<AG, NG, false>, sweep_umma_kernel<AG, NG, true>}}

static const UShape *umma_shape(int per_oct)
{
    // (angles per compute warp, compute warps per octant) for the level-symmetric sets: S2 1, S4 3, S6 6, S8 10,
    // S10 15, S12 21, S14 28, S16 36 angles per octant. Measured at S16/P5 on 256x256x64 (ms per sweep): 6 angles x 6
    // warps 9.47, 9 x 4 8.11, 12 x 3 7.43, 18 x 2 8.18; at S8/P3: 2 x 5 3.71, 5 x 2 3.78, 10 x 1 4.94 -- every warp
    // pays a fixed per-step cost (waits, arrivals, fences, its share of staging / split / read-back), so few warps with
    // many angles win until the chains get too long.
    static const UShape shapes[] = {
        USHAPE(1, 1), USHAPE(1, 3), USHAPE(2, 3), USHAPE(5, 2), USHAPE(5, 3), USHAPE(7, 3), USHAPE(14, 2), USHAPE(12, 3),
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
           up((size_t)A * 16) + up((size_t)n_mat * A * 4) + up((size_t)n_mat * 4) + up((size_t)8 * MP * 4) + up((size_t)A * DOS_TJ * 4) +
           up(64 * 8) + up(32 * 4) + 128;
}

cudaError_t dos_sweep_umma_grid(int L, int per_oct, int n_mat, int n_items, int *grid_out)
{
    const UShape *s = umma_shape(per_oct);
    if (!s) return cudaErrorInvalidValue;
    const size_t smem = umma_smem(dos_mpad(L), per_oct, n_mat);
    cudaError_t e = cudaSuccess;
    for (int v = 0; v < 2; ++v) {
        if ((e = cudaFuncSetAttribute(s->fn[v], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)) != cudaSuccess) return e;
        if (umma_realloc(s->ag, s->ng)) {     // the launch must own the registers the roles re-divide (see umma_reg_*)
            cudaFuncAttributes fa;
            if ((e = cudaFuncGetAttributes(&fa, s->fn[v])) != cudaSuccess) return e;
            if (fa.numRegs * (4 * s->ng + 4) < umma_reg_compute(s->ng) * 4 * s->ng + umma_reg_helper() * 4) return cudaErrorLaunchOutOfResources;
        }
    }
    int dev = 0, sms = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    // one CTA per SM: each allocates all 512 tensor-memory columns
    *grid_out = sms < n_items ? sms : n_items;
    return cudaSuccess;
}

cudaError_t dos_launch_sweep_umma(const SweepUArgs &a, int L, int grid, cudaStream_t st)
{
    const UShape *s = umma_shape(a.per_oct);
    if (!s) return cudaErrorInvalidValue;
    const size_t smem = umma_smem(dos_mpad(L), a.per_oct, a.n_mat);
    s->fn[a.refl ? 1 : 0]<<<grid, (4 * s->ng + 4) * 32, smem, st>>>(a);
    return cudaGetLastError();
}
