/* ewald_kernels_common.cuh -- small device helpers shared by the kernels. */
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ewald {

template <typename T> struct Num;
template <> struct Num<double> {
    typedef double2 T2;
    static __device__ __forceinline__ void sincospi_(double x, double *s, double *c) { sincospi(x, s, c); }
    static __device__ __forceinline__ double rint_(double x) { return rint(x); }
    static __device__ __forceinline__ double erfc_(double x) { return erfc(x); }
    static __device__ __forceinline__ double rsqrt_(double x) { return rsqrt(x); }
};
template <> struct Num<float> {
    typedef float2 T2;
    static __device__ __forceinline__ void sincospi_(float x, float *s, float *c) { sincospif(x, s, c); }
    static __device__ __forceinline__ float rint_(float x) { return rintf(x); }
    static __device__ __forceinline__ float erfc_(float x) { return erfcf(x); }
    static __device__ __forceinline__ float rsqrt_(float x) { return rsqrtf(x); }
};

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

/* Sum over the block in FP64; result valid in thread 0.  `red` holds >= 32 doubles. */
__device__ __forceinline__ double block_sum(double v, double *red)
{
    v = warp_sum(v);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) red[wid] = v;
    __syncthreads();
    if (wid == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        v = lane < nw ? red[lane] : 0.0;
        v = warp_sum(v);
    }
    return v;
}

/* ---- TMA bulk copy global -> shared (cp.async.bulk, SASS UBLKCP) completing on an mbarrier ---------------
 * One thread initialises the barrier (then __syncthreads), one thread issues the copy, every thread that reads the
 * data waits on the barrier's phase.  bytes: multiple of 16; source and destination 16-byte aligned. */
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void tma_barrier_init(uint64_t *bar)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(bar)) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void tma_load_1d(void *dst_smem, const void *src_gmem, unsigned bytes, uint64_t *bar)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
/* Several bulk copies on one barrier: the issuing thread announces the total once, then starts the copies
 * (each a multiple of 16 bytes, 16-byte aligned on both sides; long ones are cut into pieces of at most 32 KB). */
__device__ __forceinline__ void tma_expect(uint64_t *bar, unsigned total_bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(total_bytes) : "memory");
}
__device__ __forceinline__ void tma_copy_1d(void *dst_smem, const void *src_gmem, unsigned bytes, uint64_t *bar)
{
    constexpr unsigned PIECE = 32 * 1024;
    for (unsigned o = 0; o < bytes; o += PIECE) {
        const unsigned b = bytes - o < PIECE ? bytes - o : PIECE;
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(smem_u32(dst_smem) + o), "l"((const char *)src_gmem + o), "r"(b), "r"(smem_u32(bar)) : "memory");
    }
}
__device__ __forceinline__ void tma_wait(uint64_t *bar, unsigned parity)
{
    unsigned done;
    do {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!done);
}

/* Power table of one point for one direction: tab[n] = scale * exp(2 pi i s)^n, n = 0..nmax. */
template <typename T>
__device__ __forceinline__ void power_row(T s, T scale, int nmax, typename Num<T>::T2 *tab)
{
    typedef typename Num<T>::T2 T2;
    s -= Num<T>::rint_(s); /* exact: the phase is periodic in s */
    T sn, cs;
    Num<T>::sincospi_(2 * s, &sn, &cs);
    T2 e; e.x = scale; e.y = 0;
    tab[0] = e;
    for (int n = 1; n <= nmax; n++) {
        T2 f;
        f.x = e.x * cs - e.y * sn;
        f.y = e.x * sn + e.y * cs;
        e = f;
        tab[n] = e;
    }
}

} // namespace ewald
