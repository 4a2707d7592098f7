// dos_sweep.cu -- the S_N transport sweep (eq. 2-3) for one group and one source
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
//   moments     both contractions run on the tensor cores (mma.sync m16n8k8, 3xTF32 split, fp32 accumulate) in
//               the aux warps: M2D one step ahead of the compute warps (q_n[cell][angle] to shared memory),
//               D2M one step behind (psi_c from shared memory, summed over ALL angles of the octant, then one
//               red.global.add.v2.f32 per cell, octant and 2 moments). ncu of the FFMA version showed the two
//               contractions at 47 % of the instructions and 87 % of the shared-memory wavefronts
//               (profiles/r1c_sweep_full.md).
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

// CTA-scope release / acquire on a shared-memory word (service warp <-> compute warps)
__device__ __forceinline__ void st_release_cta(int *p, int v)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(p);
    asm volatile("st.release.cta.shared.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ int ld_acquire_cta(const int *p)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(p);
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
__device__ __forceinline__ void sts_f32(unsigned a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ void sts_s32(unsigned a, int v) { asm volatile("st.shared.s32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }

// Optional per-step timeline of one work item (option "sweep_trace_item"): every warp's lane 0 stores the SM
// clock when it starts a step (0), after its staging / M2D phase (1), after its D2M / diamond-difference phase (2)
// and when it reaches the step's barrier (3): trace[(step * 32 + warp) * 4 + k].
// Compiled in only with -DDOS_SWEEP_TRACE=1 (the test in every step costs ~4 % of the instructions).
#ifndef DOS_SWEEP_TRACE
#define DOS_SWEEP_TRACE 0
#endif
__device__ __forceinline__ void trace_mark(long long *trace, int step, int warp, int which)
{
#if DOS_SWEEP_TRACE
    if (trace && (threadIdx.x & 31) == 0) trace[(step * 32 + warp) * 4 + which] = clock64();
#else
    (void)trace; (void)step; (void)warp; (void)which;
#endif
}

// barrier of the compute warps only (the service warp never joins it)
__device__ __forceinline__ void bar_compute(int n_threads) { asm volatile("bar.sync 1, %0;" ::"r"(n_threads) : "memory"); }

__device__ __forceinline__ void st_release(int *p, int v)
{
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

__device__ __forceinline__ void red_add_v2(float *p, float a, float b)
{
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(a), "f"(b) : "memory");
}

constexpr int NT = 5;     // angle tiles (of 8) whose M2D accumulators an aux lane holds at a time
constexpr int PS = 40;    // floats per angle row of the psi_c buffer: conflict-free A-fragment loads (8 t + g)
constexpr int QS = 36;    // floats per angle row of the discrete-source buffer: conflict-free D-fragment stores

// ---- 3xTF32 tensor-core contraction (moment-to-discrete and discrete-to-moment) ----
// An fp32 value x is split into hi = tf32(x) and lo = tf32(x - hi), both exactly representable in TF32;
// a*b ~ a_lo*b_hi + a_hi*b_lo + a_hi*b_hi with fp32 accumulation. The dropped a_lo*b_lo term and the rounding of
// the lo parts are each <= 2^-22 |a||b|, the size of fp32 rounding itself.
__device__ __forceinline__ unsigned tf32_rna(float x)
{
    unsigned r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ void tf32_split(float x, unsigned &hi, unsigned &lo)
{
    hi = tf32_rna(x);
    lo = tf32_rna(x - __uint_as_float(hi));
}
// D(16x8) += A(16x8, row) B(8x8, col); lane = 4 g + t holds A (g,t) (g+8,t) (g,t+4) (g+8,t+4), B (k=t,n=g)
// (k=t+4,n=g), D (g,2t) (g,2t+1) (g+8,2t) (g+8,2t+1).
__device__ __forceinline__ void mma_tf32(float (&d)[4], const unsigned (&a)[4], unsigned b0, unsigned b1)
{
    asm("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
// The same split for the A operands in the step loop. cvt.rna.tf32.f32 has no SASS instruction on sm_100 (ptxas
// emits a 5-instruction sequence), so hi is rounded with an integer add on the bit pattern (round half away from
// zero; the inputs are finite and far from FLT_MAX) and lo = x - hi (exact) is handed to the MMA as it is: the
// tensor core drops its low 13 bits, an error <= 2^-21 |x|.
__device__ __forceinline__ void tf32_split_fast(float x, unsigned &hi, unsigned &lo)
{
    hi = (__float_as_uint(x) + 0x1000u) & 0xffffe000u;
    lo = __float_as_uint(x - __uint_as_float(hi));
}
// N independent 16x8 accumulators share one split A fragment; b[i] = (b0 hi, b1 hi, b0 lo, b1 lo). The three terms
// are issued term-major so that consecutive MMAs are independent (a dependent HMMA waits ~20 cycles), small terms first.
template <int N>
__device__ __forceinline__ void mma_3xtf32(float (&d)[N][4], const unsigned (&ah)[4], const unsigned (&al)[4], const float4 (&b)[N])
{
#pragma unroll
    for (int i = 0; i < N; ++i) mma_tf32(d[i], al, __float_as_uint(b[i].x), __float_as_uint(b[i].y));
#pragma unroll
    for (int i = 0; i < N; ++i) mma_tf32(d[i], ah, __float_as_uint(b[i].z), __float_as_uint(b[i].w));
#pragma unroll
    for (int i = 0; i < N; ++i) mma_tf32(d[i], ah, __float_as_uint(b[i].x), __float_as_uint(b[i].y));
}

// M2D of one 16-cell row tile for N consecutive 8-angle tiles: qa -> this lane's A elements of k-step 0 (row stride
// MPS), bf -> this lane's B fragments of the first angle tile ([tile][KM][32] float4), out -> this lane's D elements.
template <int MPS, int KM, int N>
__device__ __forceinline__ void m2d_tiles(const float *qa, const float4 *bf, float *out)
{
    float d[N][4];
#pragma unroll
    for (int i = 0; i < N; ++i) d[i][0] = d[i][1] = d[i][2] = d[i][3] = 0.f;
#pragma unroll
    for (int ks = 0; ks < KM; ++ks) {
        unsigned ah[4], al[4];
        const float *q0 = qa + ks * 8;
        tf32_split_fast(q0[0], ah[0], al[0]); tf32_split_fast(q0[8 * MPS], ah[1], al[1]);
        tf32_split_fast(q0[4], ah[2], al[2]); tf32_split_fast(q0[8 * MPS + 4], ah[3], al[3]);
        float4 b[N];
#pragma unroll
        for (int i = 0; i < N; ++i) b[i] = bf[(i * KM + ks) * 32];
        mma_3xtf32<N>(d, ah, al, b);
    }
#pragma unroll
    for (int i = 0; i < N; ++i) {
        float *o8 = out + i * 8 * QS;
        o8[0] = d[i][0]; o8[QS] = d[i][1]; o8[8] = d[i][2]; o8[QS + 8] = d[i][3];
    }
}

// D2M of one 16-cell row tile for the N 8-moment tiles I0..I0+N-1: pa -> this lane's A elements (psi_c) of angle
// tile 0, bf -> this lane's B fragments ([moment tile][NA][32] float4), r0 / r1 -> phi of the lane's two cells at
// moment 2 t4 (rows g8, g8 + 8); one red.global.add.v2 per (cell, 2 moments).
template <int MP, int I0, int N>
__device__ __forceinline__ void d2m_tiles(const float *pa, const float4 *bf, int NA, float *r0, float *r1, bool on0, bool on1, int t4)
{
    if constexpr (N > 0) {
    float d[N][4];
#pragma unroll
    for (int i = 0; i < N; ++i) d[i][0] = d[i][1] = d[i][2] = d[i][3] = 0.f;
#pragma unroll 1
    for (int ka = 0; ka < NA; ++ka) {
        unsigned ah[4], al[4];
        const float *p0 = pa + ka * 8 * PS;
        tf32_split_fast(p0[0], ah[0], al[0]); tf32_split_fast(p0[8], ah[1], al[1]);
        tf32_split_fast(p0[4 * PS], ah[2], al[2]); tf32_split_fast(p0[4 * PS + 8], ah[3], al[3]);
        float4 b[N];
#pragma unroll
        for (int i = 0; i < N; ++i) b[i] = bf[((I0 + i) * NA + ka) * 32];
        mma_3xtf32<N>(d, ah, al, b);
    }
#pragma unroll
    for (int i = 0; i < N; ++i)
        if ((I0 + i) * 8 + 2 * t4 < MP) {
            if (on0) red_add_v2(r0 + (I0 + i) * 8, d[i][0], d[i][1]);
            if (on1) red_add_v2(r1 + (I0 + i) * 8, d[i][2], d[i][3]);
        }
    }
}

// 16-byte asynchronous global -> shared copy that bypasses L1 (tile faces are written by other SMs
// during this launch; an L1 line could be stale)
__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
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
    float *dst0;
    int sstep, dslot, lo, hi, dist, mask;
};

struct ItemGeom {
    int o, tj, tk, id;
    bool has_y, has_z;
    const float *fy_in, *fz_in;
};

// Decode load `op` of the current item: ops [0, 32 MV) fetch 4 moments of lane c's cell, the next A
// fetch the 4 y-face inflows of angle a, the last 2A the 8 z-face inflows of angle a in two halves.
template <int MP>
__device__ __forceinline__ LoadOp make_op(int op, const Sweep2Args &p, const ItemGeom &g, float *s_q, float *s_fin)
{
    constexpr int MV = MP / 4, MPS = mps_of(MP);
    const int A = p.per_oct, nx = p.nx;
    LoadOp d;
    d.lo = 1; d.hi = 0;                      // empty window
    d.src0 = p.Q; d.dst0 = s_q; d.sstep = 0; d.dslot = 0; d.dist = DQ; d.mask = RQ - 1;
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
        d.dst0 = s_q + c * MPS + 4 * v;
        d.dslot = 32 * MPS;
    } else if (op < 32 * MV + A) {
        const int a = op - 32 * MV;
        if (g.has_y) { d.lo = 0; d.hi = nx + DOS_TK - 2; }
        d.src0 = g.fy_in + a * DOS_TK;
        d.sstep = A * DOS_TK;
        d.dst0 = s_fin + a * FINW;
        d.dslot = A * FINW; d.dist = DF; d.mask = RF - 1;
    } else {
        const int idx = op - 32 * MV - A, a = idx >> 1, h = idx & 1;
        if (g.has_z) { d.lo = 0; d.hi = nx + DOS_TJ - 2; }
        d.src0 = g.fz_in + a * DOS_TJ + 4 * h;
        d.sstep = A * DOS_TJ;
        d.dst0 = s_fin + a * FINW + DOS_TK + 4 * h;
        d.dslot = A * FINW; d.dist = DF; d.mask = RF - 1;
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
// TMAX = CTA size bound for the register budget.
template <int MP, int AG, int TMAX, int MINB>
__global__ void __launch_bounds__(TMAX, MINB) sweep_kernel(const Sweep2Args p)
{
    constexpr int MV = MP / 4, MPS = mps_of(MP), KM = (MP + 7) / 8;
    extern __shared__ float4 smem4[];
    const int A = p.per_oct, NW = p.n_warps, NX = p.n_aux;
    const int NA = (A + 7) / 8, A8 = NA * 8;                // angles in 8-wide MMA tiles
    const int NB = (NW + NX + 1) * 32;                      // threads in the per-step barrier (compute, aux, feeder)
    float *s_q = reinterpret_cast<float *>(smem4);          // [RQ][32][MPS] staged source moments (+ 8 floats of slack)
    float *s_fin = s_q + RQ * 32 * MPS + 8;                 // [RF][A][FINW] staged tile-inflow faces
    float *s_psi = s_fin + RF * A * FINW;                   // [2][A8][PS]   psi_c of the last two steps
    float *s_qd = s_psi + 2 * A8 * PS;                      // [2][A8][QS]   discrete source q_n of this and the next step
    float *s_bm = s_qd + 2 * A8 * QS;                       // [NA][KM][32][4] M2D B fragments (b0 hi, b1 hi, b0 lo, b1 lo)
    float *s_bd = s_bm + NA * KM * 128;                     // [KM][NA][32][4] D2M B fragments
    float *s_cdd = s_bd + NA * KM * 128;                    // [A][4]
    float *s_rden = s_cdd + A * 4;                          // [n_mat][A]  1 / (sigma_t + cx + cy + cz)
    float *s_sig = s_rden + p.n_mat * A;                    // [n_mat]
    int *s_mat = reinterpret_cast<int *>(s_sig + ((p.n_mat + 3) & ~3));   // [4][32] material ids of 4 steps
    __shared__ int s_item;
    __shared__ int s_done;        // steps finished by the compute/aux warps (written by one aux thread)
    __shared__ int s_allowed;     // last step whose tile-inflow faces are published upwind (service warp)

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool tick = warp == NW + NX, service = warp == NW + NX + 1, aux = warp >= NW && warp < NW + NX;
    const int jj = lane & (DOS_TJ - 1), kk = lane / DOS_TJ;
    const int skew = jj + kk;
    const int nx = p.nx, ny = p.ny, nz = p.nz;
    const int T = nx + DOS_SKEW;
    const size_t fstride_y = (size_t)(nx + DOS_FACE_PAD) * A * DOS_TK, fstride_z = (size_t)(nx + DOS_FACE_PAD) * A * DOS_TJ;

    // Everything in shared memory stays finite: the MMA tiles read padding (moments >= MP, angles >= A) against
    // zero coefficients, and 0 * garbage must be 0.
    {
        float *s_end = reinterpret_cast<float *>(s_mat + 4 * 32);
        for (float *z = s_q + tid; z < s_end; z += blockDim.x) *z = 0.f;
    }
    __syncthreads();
    for (int t = tid; t < p.n_mat; t += blockDim.x) s_sig[t] = p.sig_t[t];
    int cur_oct = -1;

    for (;;) {
        __syncthreads();                              // previous item finished with the staging buffers
        if (tid == 0) s_item = atomicAdd(p.queue, 1);
        __syncthreads();
        const int item = s_item;
        if (item >= p.n_items) break;
        const int tile_item = item / p.a_split, part = item - tile_item * p.a_split;
        const int packed = p.items[tile_item];
        ItemGeom g;
        g.o = packed & 7; g.tj = (packed >> 3) & 0x3FFF; g.tk = packed >> 17;
        g.id = ((g.o * p.ntk + g.tk) * p.ntj + g.tj) * p.a_split + part;
        g.has_y = g.tj > 0; g.has_z = g.tk > 0;
        g.fy_in = p.fy + (g.has_y ? (size_t)(g.id - p.a_split) * fstride_y : 0);
        g.fz_in = p.fz + (g.has_z ? (size_t)(g.id - p.ntj * p.a_split) * fstride_z : 0);
        const int o = g.o;
        long long *const trace = (p.trace && g.id == p.trace_item) ? p.trace : nullptr;
        if (o * 8 + part != cur_oct) {
            // tables of this CTA's angles [o][part * A, (part + 1) * A), as pre-split TF32 B fragments
            const float *m2d = p.m2d + ((size_t)o * p.per_oct_full + (size_t)part * A) * MP;
            const float *d2m = p.d2m + ((size_t)o * p.per_oct_full + (size_t)part * A) * MP;
            for (int idx = tid; idx < NA * KM * 32; idx += blockDim.x) {
                const int ln = idx & 31, tile = idx >> 5, gg = ln >> 2, tt = ln & 3;
                {   // M2D: tile (nt, ks); B[k = moment][n = angle] = m2d[angle][moment]
                    const int nt = tile / KM, ks = tile - nt * KM, a = nt * 8 + gg, m0 = ks * 8 + tt, m1 = m0 + 4;
                    const float b0 = (a < A && m0 < MP) ? m2d[a * MP + m0] : 0.f, b1 = (a < A && m1 < MP) ? m2d[a * MP + m1] : 0.f;
                    unsigned h0, l0, h1, l1;
                    tf32_split(b0, h0, l0); tf32_split(b1, h1, l1);
                    reinterpret_cast<float4 *>(s_bm)[idx] = make_float4(__uint_as_float(h0), __uint_as_float(h1), __uint_as_float(l0), __uint_as_float(l1));
                }
                {   // D2M: tile (nm, ka); B[k = angle][n = moment] = d2m[angle][moment]
                    const int nm = tile / NA, ka = tile - nm * NA, mo = nm * 8 + gg, a0 = ka * 8 + tt, a1 = a0 + 4;
                    const float b0 = (a0 < A && mo < MP) ? d2m[a0 * MP + mo] : 0.f, b1 = (a1 < A && mo < MP) ? d2m[a1 * MP + mo] : 0.f;
                    unsigned h0, l0, h1, l1;
                    tf32_split(b0, h0, l0); tf32_split(b1, h1, l1);
                    reinterpret_cast<float4 *>(s_bd)[idx] = make_float4(__uint_as_float(h0), __uint_as_float(h1), __uint_as_float(l0), __uint_as_float(l1));
                }
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
            int published = 0, spins = 0;
            for (;;) {
                const int dn = ld_acquire_cta(&s_done);
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
                        if (lane == 0) st_release_cta(&s_allowed, al);
                        spins = 0;
                    } else {
                        // watchdog: a hand-off that never arrives must not hang the GPU; the result is then
                        // invalid and dos_check / dos_dose_host report DOS_ERR_CUDA
                        if (++spins > DOS_SPIN_LIMIT) atomicExch(p.abort_flag, 1);
                        if ((spins & 255) == 0 && ld_relaxed(p.abort_flag)) {
                            avail_y = avail_z = BIG;
                            if (lane == 0) st_release_cta(&s_allowed, BIG);
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
            const LoadOp op0 = make_op<MP>(32 * MV + (lane < n_fops ? lane : 0), p, g, s_q, s_fin);
            const bool op0_on = lane < n_fops, more_ops = n_fops > 32;
            const uint8_t *mat_p = p.mat + cbase + 3 * istep;            // material of step t + 3
            const unsigned mat_w = smem_addr(s_mat + lane);
            auto mat_of = [&](int s, const uint8_t *q) -> int {
                return ((unsigned)(s - t_lo) < (unsigned)nx) ? (int)__ldg(q) : 0;
            };
            __syncthreads();                          // S2: s_done, s_allowed in place
            int allowed_c = -1;
            auto issue_one = [&](const LoadOp &d, int tau) {
                const int s = tau + DF;
                if (s >= d.lo && s <= d.hi) {
                    while (allowed_c < s) {           // wait until the upwind tiles have published step s
                        allowed_c = ld_acquire_cta(&s_allowed);
                        if (allowed_c < s) __nanosleep(DOS_POLL_NS);
                    }
                    cp_async16(d.dst0 + (s & d.mask) * d.dslot, d.src0 + (long long)s * d.sstep);
                }
            };
            auto issue_round = [&](int tau) {         // round tau fetches the tile-inflow faces of step tau + DF
                if (op0_on) issue_one(op0, tau);
                if (more_ops)
                    for (int f = lane + 32; f < n_fops; f += 32) issue_one(make_op<MP>(32 * MV + f, p, g, s_q, s_fin), tau);
                cp_async_commit();
            };
            for (int tau = -DF; tau < 0; ++tau) issue_round(tau);
            sts_s32(mat_w, mat_of(0, mat_p - 3 * istep));
            sts_s32(mat_w + 128, mat_of(1, mat_p - 2 * istep));
            int reg_m = mat_of(2, mat_p - istep);
            cp_async_wait<DF - 1>();
            bar_compute(NB);                          // S3a
            bar_compute(NB);                          // S3b: step 0's staged data visible to every warp
#pragma unroll 1
            for (int t = 0; t < T; ++t) {
                trace_mark(trace, t, warp, 0);
                issue_round(t);
                sts_s32(mat_w + ((t + 2) & 3) * 128, reg_m);
                reg_m = mat_of(t + 3, mat_p);
                mat_p += istep;
                cp_async_wait<DF - 1>();              // step t + 1's faces complete (this thread's copies)
                trace_mark(trace, t, warp, 3);
                bar_compute(NB);                      // B_t: ... visible to all; every face store of step t precedes it
                if (lane == 0) st_release_cta(&s_done, t + 1);
            }
            continue;
        }

        if (aux) {
            // ------- aux warps: staging of the source moments, M2D of the next step, D2M of the previous step -------
            // Both contractions run on the tensor cores as 3xTF32 m16n8k8 MMAs over the step's 32 cells (two 16-row
            // tiles; row r of tile m is lane-cell 16 m + r of the compute warps, i.e. (jj, kk) = (r & 7, 2 m + r / 8)):
            //   M2D  q[cell][angle]  = sum_lm Q[cell][lm] (2l+1) Y_lm(angle)   A = staged moments, B = s_bm
            //   D2M  dphi[cell][lm]  = sum_a psi_c[cell][a] w_a Y_lm(a)         A = s_psi,          B = s_bd
            // A unit = one contraction for one 16-cell row tile and half of the column tiles (the A fragments are
            // loaded and split once per k-step and reused for the unit's column tiles): 8 units.
            const int xw = warp - NW, xt = tid - NW * 32, NXT = NX * 32;
            const int n_ops = 32 * MV;                                   // Q copies; the feeder warp does the faces
            const LoadOp op0 = make_op<MP>(xt < n_ops ? xt : 0, p, g, s_q, s_fin);
            const LoadOp op1 = make_op<MP>(xt + NXT < n_ops ? xt + NXT : 0, p, g, s_q, s_fin);
            const bool op0_on = xt < n_ops, op1_on = xt + NXT < n_ops, more_ops = n_ops > 2 * NXT;
            const int g8 = lane >> 2, t4 = lane & 3;
            // this lane's 4 D-fragment rows are the cells (jj = g8, kk = 0..3): pointer to phi of the row's cell at
            // step 0 (advanced by istep * MP floats per step) and first active step
            float *phi_row[4];
            int tlo_row[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const int jpr = g.tj * DOS_TJ + g8, kpr = g.tk * DOS_TK + r;
                const bool vr = jpr < ny && kpr < nz;
                const int jr = (o & 2) ? ny - 1 - jpr : jpr, kr = (o & 4) ? nz - 1 - kpr : kpr;
                const long long c0 = vr ? ((long long)kr * ny + jr) * nx + ((o & 1) ? nx - 1 : 0) - (long long)istep * (g8 + r) : 0;
                phi_row[r] = p.phi + c0 * MP + 2 * t4;
                tlo_row[r] = vr ? g8 + r : BIG;
            }
            const int phi_inc = istep * MP;
            __syncthreads();                          // S2: octant tables in place
            auto issue_one = [&](const LoadOp &d, int tau) {
                const int s = tau + DQ;
                if (s >= d.lo && s <= d.hi) cp_async16(d.dst0 + (s & d.mask) * d.dslot, d.src0 + (long long)s * d.sstep);
            };
            auto issue_round = [&](int tau) {         // round tau fetches the source moments of step tau + DQ
                if (op0_on) issue_one(op0, tau);
                if (op1_on) issue_one(op1, tau);
                if (more_ops)
                    for (int op = xt + 2 * NXT; op < n_ops; op += NXT) issue_one(make_op<MP>(op, p, g, s_q, s_fin), tau);
                cp_async_commit();
            };
            // moment-to-discrete of step s for the 16 cells of row tile m, angle tiles [n_lo, n_hi) -> s_qd[s & 1]
            auto m2d_unit = [&](int s, int m, int n_lo, int n_hi) {
                const float *qa = s_q + (s & (RQ - 1)) * (32 * MPS) + (16 * m + g8) * MPS + t4;
                const float4 *bf = reinterpret_cast<const float4 *>(s_bm) + lane;
                float *out = s_qd + (s & 1) * (A8 * QS) + 2 * t4 * QS + 16 * m + g8;
                for (int nt0 = n_lo; nt0 < n_hi; nt0 += NT) {      // uniform dispatch: no predicated MMAs
                    const float4 *b0 = bf + nt0 * KM * 32;
                    float *o0 = out + nt0 * 8 * QS;
                    switch (min(n_hi - nt0, NT)) {
                        case 1: m2d_tiles<MPS, KM, 1>(qa, b0, o0); break;
                        case 2: m2d_tiles<MPS, KM, 2>(qa, b0, o0); break;
                        case 3: m2d_tiles<MPS, KM, 3>(qa, b0, o0); break;
                        case 4: m2d_tiles<MPS, KM, 4>(qa, b0, o0); break;
                        default: m2d_tiles<MPS, KM, 5>(qa, b0, o0); break;
                    }
                }
            };
            // discrete-to-moment of step s for the 16 cells of row tile m, first (h = 0) or second half of the moment tiles
            auto d2m_unit = [&](int s, int m, int h) {
                const float *pa = s_psi + (s & 1) * (A8 * PS) + t4 * PS + 16 * m + g8;
                const float4 *bf = reinterpret_cast<const float4 *>(s_bd) + lane;
                const int tl0 = m ? tlo_row[2] : tlo_row[0], tl1 = m ? tlo_row[3] : tlo_row[1];
                const bool on0 = (unsigned)(s - tl0) < (unsigned)nx, on1 = (unsigned)(s - tl1) < (unsigned)nx;
                float *r0 = (m ? phi_row[2] : phi_row[0]) + (long long)s * phi_inc;
                float *r1 = (m ? phi_row[3] : phi_row[1]) + (long long)s * phi_inc;
                constexpr int K0 = (KM + 1) / 2;
                if (h < 0) d2m_tiles<MP, 0, KM>(pa, bf, NA, r0, r1, on0, on1, t4);
                else if (h == 0) d2m_tiles<MP, 0, K0>(pa, bf, NA, r0, r1, on0, on1, t4);
                else d2m_tiles<MP, K0, KM - K0>(pa, bf, NA, r0, r1, on0, on1, t4);
            };
            // 8 units: u = kind (0 M2D, 1 D2M) * 4 + row tile m * 2 + half h of the column tiles, dealt round-robin to
            // the aux warps; with 4 or fewer aux warps the two halves are one unit (u odd is empty).
            const int NAh = (NA + 1) / 2;
            const bool halves = NX > 4;
            auto run_unit = [&](int u, int t) {
                const int m = (u >> 1) & 1, h = u & 1;
                if (!halves && h) return;
                if (u < 4) {
                    if (t + 1 < T) m2d_unit(t + 1, m, h ? NAh : 0, (h || !halves) ? NA : NAh);
                } else if (t > 0) {
                    d2m_unit(t - 1, m, halves ? h : -1);
                }
            };
            const int u0 = halves ? xw : 2 * xw, du = halves ? NX : 2 * NX;
            for (int tau = -DQ; tau < 0; ++tau) issue_round(tau);
            cp_async_wait<DF - 1>();
            bar_compute(NB);                          // S3a: the first steps' staged moments visible to the aux warps
            for (int u = u0; u < 4; u += du) run_unit(u, -1);
            bar_compute(NB);                          // S3b: q_n of step 0 visible to the compute warps

#pragma unroll 1
            for (int t = 0; t < T; ++t) {
                trace_mark(trace, t, warp, 0);
                issue_round(t);
                trace_mark(trace, t, warp, 1);
                for (int u = u0; u < 8; u += du) run_unit(u, t);
                trace_mark(trace, t, warp, 2);
                cp_async_wait<DF - 1>();              // staged moments up to step t + DQ - DF + 1 complete (this thread's copies)
                trace_mark(trace, t, warp, 3);
                bar_compute(NB);                      // B_t: ... and visible to all
            }
            for (int u = u0; u < 8; u += du)
                if (u >= 4) run_unit(u, T);
            continue;
        }

        // ---------------- compute warps: diamond difference, face hand-off ----------------
        const int a0 = warp * AG;
        const bool in_y = jj == 0, in_z = kk == 0;
        const bool has_y = g.has_y, has_z = g.has_z;
        const bool store_y = valid && jj == DOS_TJ - 1 && g.tj < p.ntj - 1;
        const bool store_z = valid && kk == DOS_TK - 1 && g.tk < p.ntk - 1;
        // running pointers, advanced once per step
        float *fy_st = p.fy + (size_t)g.id * fstride_y + kk + ((long long)(1 - DOS_TJ) * A + a0) * DOS_TK;
        float *fz_st = p.fz + (size_t)g.id * fstride_z + jj + ((long long)(1 - DOS_TK) * A + a0) * DOS_TJ;
        const int fy_inc = A * DOS_TK, fz_inc = A * DOS_TJ;
        const unsigned fin_y = smem_addr(s_fin + a0 * FINW + kk), fin_z = smem_addr(s_fin + a0 * FINW + DOS_TK + jj);
        const unsigned psi_w = smem_addr(s_psi + a0 * PS + lane);
        const unsigned qd_r = smem_addr(s_qd + a0 * QS + lane);
        const unsigned rden_a = smem_addr(s_rden + a0), sig_a = smem_addr(s_sig), mat_r = smem_addr(s_mat + lane);
        const int fin_slot = A * FINW * 4, psi_slot = A8 * PS * 4, qd_slot = A8 * QS * 4, A4 = A * 4;

        float ccx[AG], ccy[AG], ccz[AG];
        __syncthreads();                              // S2: octant tables, s_done, s_allowed in place
#pragma unroll
        for (int r = 0; r < AG; ++r) {
            ccx[r] = s_cdd[(a0 + r) * 4 + 0]; ccy[r] = s_cdd[(a0 + r) * 4 + 1]; ccz[r] = s_cdd[(a0 + r) * 4 + 2];
        }
        float px[AG], oy[AG], oz[AG];
#pragma unroll
        for (int r = 0; r < AG; ++r) px[r] = oy[r] = oz[r] = 0.f;
        bar_compute(NB);                              // S3a
        bar_compute(NB);                              // S3b: step 0's staged data and q_n visible

#pragma unroll 1
        for (int t = 0; t < T; ++t) {
            trace_mark(trace, t, warp, 0);
            const bool act = (unsigned)(t - t_lo) < (unsigned)nx;
            const int m0 = lds_s32(mat_r + (t & 3) * 128);
            // discrete source of this lane's cell for the warp's AG angles (M2D done by the aux warps one step ahead)
            float q[AG];
#pragma unroll
            for (int r = 0; r < AG; ++r) q[r] = lds_f32(qd_r + (t & 1) * qd_slot + r * (QS * 4));

            trace_mark(trace, t, warp, 1);
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
                    if (store_y) __stcg(fy_st + r * DOS_TK, oyr);
                    if (store_z) __stcg(fz_st + r * DOS_TJ, ozr);
                }
                sts_f32(pso + r * (PS * 4), pc);
            }
            fy_st += fy_inc; fz_st += fz_inc;
            trace_mark(trace, t, warp, 2);
            trace_mark(trace, t, warp, 3);
            bar_compute(NB);                          // B_t
        }
    }
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side: choice of angles per warp, occupancy-sized persistent grid, template dispatch
// ------------------------------------------------------------------------------------------------
typedef void (*sweep_fn)(const Sweep2Args);

// variant 0: up to 16 warps, 1 CTA per SM (128 registers); 1: up to 20 warps (102 registers); 2: up to 16 warps,
// 2 CTAs per SM (64 registers), for few moments per cell where the register cap costs only a few spills
template <int MP, int AG>
static sweep_fn pick_var(int var)
{
    if (var == 1) return sweep_kernel<MP, AG, 640, 1>;
    if (var == 2) return MP <= 16 ? sweep_kernel<MP <= 16 ? MP : 4, AG, 512, 2> : nullptr;
    return sweep_kernel<MP, AG, 512, 1>;
}

template <int MP>
static sweep_fn pick_ag(int ag, int var)
{
    switch (ag) {
        case 1: return pick_var<MP, 1>(var);
        case 2: return pick_var<MP, 2>(var);
        case 3: return pick_var<MP, 3>(var);
        case 4: return pick_var<MP, 4>(var);
    }
    return nullptr;
}

static int g_two_per_sm = 0;     // allow the 2-CTAs-per-SM variant (option "sweep_two_per_sm")
void dos_sweep_set_two_per_sm(int on) { g_two_per_sm = on; }

// n_items decides between variants 0 and 2: two CTAs per SM pay off when there are more work items than SMs
static sweep_fn pick(int L, int ag, int per_oct, int n_aux, int n_items)
{
    const int warps = per_oct / ag + n_aux + 2, MP = dos_mpad(L);
    int sms = 148, dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int var = warps > 16 ? 1 : ((g_two_per_sm && MP <= 16 && n_items > sms) ? 2 : 0);
    switch (MP) {
        case 4: return pick_ag<4>(ag, var);
        case 12: return pick_ag<12>(ag, var);
        case 16: return pick_ag<16>(ag, var);
        case 28: return pick_ag<28>(ag, var);
        case 36: return pick_ag<36>(ag, var);
    }
    return nullptr;
}

static size_t sweep_smem(int L, int per_oct, int n_mat)
{
    const int MP = dos_mpad(L), MPS = mps_of(MP), A = per_oct, KM = (MP + 7) / 8, NA = (A + 7) / 8, A8 = NA * 8;
    const size_t floats = (size_t)RQ * 32 * MPS + 8 + (size_t)RF * A * FINW + (size_t)2 * A8 * PS + (size_t)2 * A8 * QS +
                          (size_t)2 * NA * KM * 128 + (size_t)4 * A + (size_t)n_mat * A + ((n_mat + 3) & ~3) + 4 * 32 + 4;
    return sizeof(float) * floats;
}

int dos_sweep_trace_compiled() { return DOS_SWEEP_TRACE; }

// Angles per warp AG (1..4, must divide the octant's angle count A; the CTA has A/AG compute warps, up to 4 aux
// warps, a feeder and a service warp, at most 20 warps). Default: the smallest AG with at most 10 compute warps (so
// that 8 aux warps fit) -- few angles per warp keep the per-step dependent chain short (S2: 1x1, S4: 3x1, S6: 6x1,
// S8: 10x1, S12: 7x3, S16: 9x4). `prefer` > 0 overrides when it is admissible (at most 14 compute warps).
// Aux warps (staging + the two tensor-core contractions): the contraction work comes in 4 units (M2D and D2M x
// two 16-cell row tiles), or 8 when each is split in two halves of its column tiles. Default 4 aux warps, one unit
// each (measured faster than 8 half units on configs 2 and 3). `prefer` > 0 overrides (1, 2, 4 or 8).
int dos_sweep_aux_warps(int per_oct, int L, int ag, int prefer)
{
    (void)L;
    const int nw = per_oct / ag;
    if (prefer >= 1) return prefer >= 8 ? 8 : (prefer >= 4 ? 4 : (prefer >= 2 ? 2 : 1));
    return nw + 4 + 2 <= 20 ? 4 : 2;
}

int dos_sweep_angles_per_warp(int per_oct, int L, int prefer)
{
    (void)L;
    if (prefer >= 1 && prefer <= 4 && per_oct % prefer == 0 && per_oct / prefer <= 14) return prefer;
    for (int ag = 1; ag <= 4; ++ag)
        if (per_oct % ag == 0 && per_oct / ag <= 10) return ag;
    for (int ag = 1; ag <= 4; ++ag)
        if (per_oct % ag == 0 && per_oct / ag <= 14) return ag;
    return 0;
}

cudaError_t dos_sweep_grid(int L, int ag, int n_aux, int per_oct, int n_mat, int n_items, int *grid_out)
{
    sweep_fn f = pick(L, ag, per_oct, n_aux, n_items);
    if (!f) return cudaErrorInvalidValue;
    const size_t smem = sweep_smem(L, per_oct, n_mat);
    cudaError_t e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
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

cudaError_t dos_launch_sweep(const Sweep2Args &a, int L, int ag, int grid, cudaStream_t s)
{
    sweep_fn f = pick(L, ag, a.per_oct, a.n_aux, a.n_items);
    if (!f) return cudaErrorInvalidValue;
    const size_t smem = sweep_smem(L, a.per_oct, a.n_mat);
    f<<<grid, (a.n_warps + a.n_aux + 2) * 32, smem, s>>>(a);
    return cudaGetLastError();
}
