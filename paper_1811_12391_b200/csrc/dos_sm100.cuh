// dos_sm100.cuh -- thin inline-PTX wrappers of the sm_100a features the sweep uses: mbarrier, bulk asynchronous
// copies (TMA unit, cp.async.bulk), tcgen05 (TMEM allocation, tcgen05.mma kind::tf32, tcgen05.ld / tcgen05.st,
// tcgen05.commit) and the fences between the generic and asynchronous proxies. CUDA path only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sm100 {

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

// ---- mbarrier (shared::cta, 64-bit) ----
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_init_fence() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// Up to `tries` polls in a three-instruction loop; each poll may suspend the thread for up to ~`hint_ns` (the
// hardware wakes it when the phase completes), so a waiting warp costs next to no issue slots. Returns 1 on success.
__device__ __forceinline__ unsigned mbar_wait_some(uint64_t *bar, unsigned parity, unsigned tries, unsigned hint_ns)
{
    unsigned ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t.reg .u32 n;\n\tmov.u32 n, %3;\n"
        "W_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %4;\n\t@p bra D_%=;\n\t"
        "sub.u32 n, n, 1;\n\tsetp.ne.u32 p, n, 0;\n\t@p bra W_%=;\n\tmov.u32 %0, 0;\n\tbra E_%=;\n"
        "D_%=:\n\tmov.u32 %0, 1;\nE_%=:\n\t}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity), "r"(tries), "r"(hint_ns)
        : "memory");
    return ok;
}
// 16-byte asynchronous copy global -> shared that bypasses L1 (LDGSTS) and an mbarrier arrival that fires when all of
// this thread's earlier cp.async have landed (no increment of the pending count: the init count covers it)
__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gmem_src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_mbar_arrive(uint64_t *bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, unsigned parity)
{
    unsigned ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
                 : "=r"(ok)
                 : "r"(smem_u32(bar)), "r"(parity)
                 : "memory");
    return ok != 0;
}

// ---- bulk asynchronous copy global -> shared (TMA unit; SASS UBLKCP), completion counted in bytes on an mbarrier ----
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gmem_src, unsigned bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// generic-proxy accesses before this fence are ordered before later asynchronous-proxy accesses (UMMA operand reads of
// shared memory, bulk copies) and vice versa
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }

// ---- tensor memory ----
__device__ __forceinline__ void tmem_alloc_512(unsigned *smem_result)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(smem_result)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_512(unsigned taddr)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(taddr) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// tcgen05.ld / tcgen05.st, shape 32x32b: thread l of the warp accesses TMEM lane (32 * (warp % 4) + l), N consecutive
// 32-bit columns starting at the column of `taddr` (whose lane field must be the warp's quarter base).
template <int N>
__device__ __forceinline__ void tmem_ld(unsigned taddr, float *v);
template <>
__device__ __forceinline__ void tmem_ld<1>(unsigned taddr, float *v)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=f"(v[0]) : "r"(taddr));
}
template <>
__device__ __forceinline__ void tmem_ld<2>(unsigned taddr, float *v)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];" : "=f"(v[0]), "=f"(v[1]) : "r"(taddr));
}
template <>
__device__ __forceinline__ void tmem_ld<4>(unsigned taddr, float *v)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];" : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]) : "r"(taddr));
}
template <>
__device__ __forceinline__ void tmem_ld<8>(unsigned taddr, float *v)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7])
                 : "r"(taddr));
}
template <>
__device__ __forceinline__ void tmem_ld<16>(unsigned taddr, float *v)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]), "=f"(v[8]), "=f"(v[9]),
                   "=f"(v[10]), "=f"(v[11]), "=f"(v[12]), "=f"(v[13]), "=f"(v[14]), "=f"(v[15])
                 : "r"(taddr));
}
template <int N>
__device__ __forceinline__ void tmem_st(unsigned taddr, const float *v);
template <>
__device__ __forceinline__ void tmem_st<1>(unsigned taddr, const float *v)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(taddr), "f"(v[0]) : "memory");
}
template <>
__device__ __forceinline__ void tmem_st<2>(unsigned taddr, const float *v)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1,%2};" ::"r"(taddr), "f"(v[0]), "f"(v[1]) : "memory");
}
template <>
__device__ __forceinline__ void tmem_st<4>(unsigned taddr, const float *v)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" ::"r"(taddr), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]) : "memory");
}
template <>
__device__ __forceinline__ void tmem_st<8>(unsigned taddr, const float *v)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(taddr), "f"(v[0]), "f"(v[1]), "f"(v[2]),
                 "f"(v[3]), "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7])
                 : "memory");
}
// N values as the largest power-of-two pieces (N <= 16)
template <int N>
__device__ __forceinline__ void tmem_ld_n(unsigned taddr, float *v)
{
    if constexpr (N >= 16) { tmem_ld<16>(taddr, v); if constexpr (N > 16) tmem_ld_n<N - 16>(taddr + 16, v + 16); }
    else if constexpr (N >= 8) { tmem_ld<8>(taddr, v); if constexpr (N > 8) tmem_ld_n<N - 8>(taddr + 8, v + 8); }
    else if constexpr (N >= 4) { tmem_ld<4>(taddr, v); if constexpr (N > 4) tmem_ld_n<N - 4>(taddr + 4, v + 4); }
    else if constexpr (N >= 2) { tmem_ld<2>(taddr, v); if constexpr (N > 2) tmem_ld_n<N - 2>(taddr + 2, v + 2); }
    else if constexpr (N == 1) { tmem_ld<1>(taddr, v); }
}
template <int N>
__device__ __forceinline__ void tmem_st_n(unsigned taddr, const float *v)
{
    if constexpr (N >= 8) { tmem_st<8>(taddr, v); if constexpr (N > 8) tmem_st_n<N - 8>(taddr + 8, v + 8); }
    else if constexpr (N >= 4) { tmem_st<4>(taddr, v); if constexpr (N > 4) tmem_st_n<N - 4>(taddr + 4, v + 4); }
    else if constexpr (N >= 2) { tmem_st<2>(taddr, v); if constexpr (N > 2) tmem_st_n<N - 2>(taddr + 2, v + 2); }
    else if constexpr (N == 1) { tmem_st<1>(taddr, v); }
}

// ---- UMMA (tcgen05.mma) ----
// Shared-memory operand descriptor, no swizzle, K-major: element (row r, 16-byte chunk c of K) of the operand sits at
// start + (r / 8) * sbo + c * lbo + (r % 8) * 16 bytes (8 x 16-byte core matrices).
__host__ __device__ __forceinline__ uint64_t umma_smem_desc(unsigned smem_addr, unsigned lbo_bytes, unsigned sbo_bytes)
{
    return (uint64_t)((smem_addr >> 4) & 0x3FFF) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32) | ((uint64_t)1 << 46);
}
// Instruction descriptor of kind::tf32: fp32 accumulate, both operands TF32 and K-major, D is M x N.
__host__ __device__ __forceinline__ unsigned umma_idesc_tf32(int M, int N)
{
    return (1u << 4) | (2u << 7) | (2u << 10) | ((unsigned)(N >> 3) << 17) | ((unsigned)(M >> 4) << 24);
}
// D[tmem] (+)= A[smem] B[smem]; one K step of 8 (32 bytes per row). Issued by ONE thread.
__device__ __forceinline__ void umma_ss(unsigned d_tmem, uint64_t a_desc, uint64_t b_desc, unsigned idesc, unsigned accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(d_tmem),
                 "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
                 : "memory");
}
// D[tmem] (+)= A[tmem] B[smem]: A row i in TMEM lane i, its K values in consecutive 32-bit columns from a_tmem.
__device__ __forceinline__ void umma_ts(unsigned d_tmem, unsigned a_tmem, uint64_t b_desc, unsigned idesc, unsigned accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}\n" ::"r"(d_tmem),
                 "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
                 : "memory");
}
// The same, issued under a predicate INSIDE the asm block (`on` is true in exactly one lane of a converged warp): a C++
// `if (leader)` around a uniform-datapath instruction makes the compiler wrap it in an ELECT / BRA.U.ANY loop.
__device__ __forceinline__ void umma_ss_if(unsigned on, unsigned d_tmem, uint64_t a_desc, uint64_t b_desc, unsigned idesc, unsigned accumulate)
{
    asm volatile("{\n\t.reg .pred p, e;\n\tsetp.ne.b32 e, %5, 0;\n\tsetp.ne.b32 p, %4, 0;\n\t@e tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(d_tmem),
                 "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate), "r"(on)
                 : "memory");
}
__device__ __forceinline__ void umma_ts_if(unsigned on, unsigned d_tmem, unsigned a_tmem, uint64_t b_desc, unsigned idesc, unsigned accumulate)
{
    asm volatile("{\n\t.reg .pred p, e;\n\tsetp.ne.b32 e, %5, 0;\n\tsetp.ne.b32 p, %4, 0;\n\t@e tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}\n" ::"r"(d_tmem),
                 "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate), "r"(on)
                 : "memory");
}
__device__ __forceinline__ void umma_commit_if(unsigned on, uint64_t *bar)
{
    asm volatile("{\n\t.reg .pred e;\n\tsetp.ne.b32 e, %1, 0;\n\t@e tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n\t}\n" ::"r"(smem_u32(bar)), "r"(on)
                 : "memory");
}
// the mbarrier gets one arrival when every tcgen05.mma issued so far by this thread has completed
__device__ __forceinline__ void umma_commit(uint64_t *bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// warp-group register re-allocation (all warps of an aligned group of 4 must execute the same one)
template <int N>
__device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N>
__device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
__device__ __forceinline__ bool elect_one()
{
    unsigned e;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}\n" : "=r"(e));
    return e != 0;
}

}  // namespace sm100
