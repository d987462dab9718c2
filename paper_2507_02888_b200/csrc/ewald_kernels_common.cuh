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
