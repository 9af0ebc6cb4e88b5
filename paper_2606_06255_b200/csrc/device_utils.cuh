// device_utils.cuh -- PTX wrappers and the few arithmetic helpers shared by the sampling kernels
// (sample_kernel.cu: one exchange per pick; sample_batched.cu: exact batched picking).
// Nothing here is used by, or taken from, oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace rfps {

constexpr unsigned FULL = 0xffffffffu;
constexpr unsigned F32_INF_BITS = 0x7f800000u;
constexpr unsigned F32_NAN_BITS = 0x7fc00000u;

// --------------------------------------------------------------------------------------------
// cluster / DSMEM / mbarrier (sm_90+; compiled for sm_100a)
// --------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned cluster_ctarank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned cluster_nctarank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
    return r;
}
// full cluster barrier with release/acquire semantics at cluster scope (orders shared::cluster AND
// global accesses of every thread of the cluster)
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cta address of this CTA -> shared::cluster address of the same variable in CTA `rank`
__device__ __forceinline__ unsigned mapa(unsigned local_addr, unsigned rank)
{
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_addr), "r"(rank));
    return r;
}
__device__ __forceinline__ unsigned ld_dsmem_u32(unsigned addr)
{
    unsigned v;
    asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ uint4 ld_dsmem_v4(unsigned addr)
{
    uint4 v;
    asm volatile("ld.shared::cluster.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void st_dsmem_u32(unsigned addr, unsigned v)
{
    asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned atom_add_dsmem_u32(unsigned addr, unsigned v)
{
    unsigned old;
    asm volatile("atom.shared::cluster.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(addr), "r"(v) : "memory");
    return old;
}
// release store to this CTA's own shared memory / acquire load from a peer's, both at cluster scope:
// a one-way message channel between CTAs of a cluster without a cluster barrier
__device__ __forceinline__ void st_release_cluster_u32(unsigned local_addr, unsigned v)
{
    asm volatile("st.release.cluster.shared::cta.u32 [%0], %1;" ::"r"(local_addr), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned ld_acquire_cluster_u32(unsigned cluster_addr)
{
    unsigned v;
    asm volatile("ld.acquire.cluster.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(cluster_addr) : "memory");
    return v;
}
// the same one-way channel through global memory at gpu scope (CTAs that are not in one cluster)
__device__ __forceinline__ void st_release_gpu_u32(unsigned *p, unsigned v)
{
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned ld_acquire_gpu_u32(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_gpu_add_u32(unsigned *p, unsigned v)
{
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void st_release_gpu_u64(unsigned long long *p, unsigned long long v)
{
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_acquire_gpu_u64(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_gpu_add_u64(unsigned long long *p, unsigned long long v)
{
    asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// release-add on a peer's shared memory, acquire load from this CTA's own shared memory
__device__ __forceinline__ void red_release_cluster_add_u32(unsigned cluster_addr, unsigned v)
{
    asm volatile("red.release.cluster.shared::cluster.add.u32 [%0], %1;" ::"r"(cluster_addr), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned ld_acquire_cluster_local_u32(unsigned local_addr)
{
    unsigned v;
    asm volatile("ld.acquire.cluster.shared::cta.u32 %0, [%1];" : "=r"(v) : "r"(local_addr) : "memory");
    return v;
}
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra WAIT_DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "WAIT_DONE:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void st_async_v4(unsigned remote_addr, unsigned a, unsigned b, unsigned c, unsigned d,
                                            unsigned remote_bar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.b32 [%0], {%1, %2, %3, %4}, [%5];" ::"r"(
                     remote_addr), "r"(a), "r"(b), "r"(c), "r"(d), "r"(remote_bar) : "memory");
}
// named barrier among `nthreads` threads of the CTA (id 1..15; id 0 is __syncthreads)
__device__ __forceinline__ void named_bar_sync(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// --------------------------------------------------------------------------------------------
// keys: (fp32 bits of d2, 0xFFFFFFFF - original index); unsigned lexicographic max = "largest
// distance, ties to the lowest original index" (Alg. 3's (d, -i_orig))
// --------------------------------------------------------------------------------------------
// max of a (hi, lo) key over the warp; returns the winning lane (lowest lane on a full tie)
__device__ __forceinline__ int warp_argmax_key(unsigned hi, unsigned lo, unsigned &mhi, unsigned &mlo)
{
    mhi = __reduce_max_sync(FULL, hi);
    mlo = __reduce_max_sync(FULL, hi == mhi ? lo : 0u);
    unsigned win = __ballot_sync(FULL, hi == mhi && lo == mlo);
    return __ffs(win) - 1;
}

// the library's one distance expression: ((dx*dx + dy*dy) + dz*dz), every operation rounded to
// nearest, never contracted to FMA (BASELINE.json north_star)
__device__ __forceinline__ float d2_rn(float x, float y, float z, float sx, float sy, float sz)
{
    const float dx = __fsub_rn(x, sx), dy = __fsub_rn(y, sy), dz = __fsub_rn(z, sz);
    return __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
}

// prune threshold of a voxel from its Dist_v and radius: the voxel is pruned iff d2(s,c) >= thr.
// thr >= (sqrt(Dv)*(1+3u) + R)^2 * (1+6u) over the reals (u = 2^-24), see DESIGN.md section 4.
__device__ __forceinline__ float prune_threshold(unsigned dv_bits, float R)
{
    if (dv_bits == 0u) return 0.0f;   // Dist_v == +0: the strict '<' of Eq. 2 can never fire
    const float q = __fadd_rn(__fmul_rn(__fsqrt_rn(__uint_as_float(dv_bits)), 1.0f + 0x1p-20f), 0x1p-40f);
    const float a = __fadd_rn(q, R);
    const float t = __fmul_rn(__fmul_rn(a, a), 1.0f + 0x1p-18f);
    return (t < __uint_as_float(F32_INF_BITS)) ? t : __uint_as_float(F32_NAN_BITS);   // inf -> NaN: never prune
}

}  // namespace rfps
