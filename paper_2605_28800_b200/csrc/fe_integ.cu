// fe_integ.cu -- array kernel of the adaptive integrator:
//   k_rk45_final  y5 = P + sum_j b5_j k_j,  err = max |sum_j d_j k_j|   (Cash-Karp 5th-order solution + embedded error)
// A plain streaming pass (HBM bound).  The right-hand sides and every other stage combination of RK45 and AB3M2 come
// from the fused local step's epilogue (fe_local.cu: LocalArgs::kOut / lk / lc).
#include "fe_internal.h"

namespace fe {

// max that keeps a NaN once it has seen one (fmax would return the other operand and hide a blown-up cell)
__device__ __forceinline__ double nanmax(double m, double v) { return (v > m || v != v) ? v : m; }

template <typename T>
__global__ void __launch_bounds__(256) k_rk45_final(T* __restrict__ y5, const T* __restrict__ P, LinArgs b5, LinArgs d,
                                                    int64_t n, unsigned long long* __restrict__ err_bits)
{
    double m = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        T v = P[i], e = (T)0;
#pragma unroll
        for (int j = 0; j < 6; ++j) {
            const T kj = static_cast<const T*>(b5.k[j])[i];
            if (b5.c[j] != 0.0) v = v + (T)b5.c[j] * kj;
            e = e + (T)d.c[j] * kj;
        }
        y5[i] = v;
        m = nanmax(m, fabs((double)e));
    }
    for (int o = 16; o > 0; o >>= 1) m = nanmax(m, __shfl_down_sync(0xffffffffu, m, o));
    __shared__ double red[8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) red[warp] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) m = nanmax(m, red[w]);
        // non-negative doubles order like their bit patterns; NaN (all-ones exponent, non-zero mantissa) sorts above
        // +inf, so a non-finite error estimate reaches the host and rejects the step
        atomicMax(err_bits, (unsigned long long)__double_as_longlong(m));
    }
}

template <typename T>
cudaError_t launch_rk45_final(T* y5, const T* P, const LinArgs& b5, const LinArgs& d, int64_t n, double* err, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(err, 0, sizeof(double), st);
    if (e != cudaSuccess) return e;
    const int grid = (int)((n + 255) / 256 < 148 * 16 ? (n + 255) / 256 : 148 * 16);
    k_rk45_final<T><<<grid, 256, 0, st>>>(y5, P, b5, d, n, reinterpret_cast<unsigned long long*>(err));
    return cudaGetLastError();
}

template cudaError_t launch_rk45_final<double>(double*, const double*, const LinArgs&, const LinArgs&, int64_t, double*, cudaStream_t);
template cudaError_t launch_rk45_final<float>(float*, const float*, const LinArgs&, const LinArgs&, int64_t, double*, cudaStream_t);

}  // namespace fe
