// bench_peaks.cu -- HARNESS kernels of bench.py, built into their own library (libfe_peaks.so), never linked
// into libfe_b200 and never on the product path:
//   fe_peak_fp64   issue rate of the fp64 pipe (dependent DFMA chains, enough warps to cover the latency),
//   fe_peak_lds    shared-memory read bandwidth (conflict-free 128-bit loads),
//   fe_peak_l2     read bandwidth of a buffer that fits in L2,
//   fe_bench_kmul  the fused 6-component k-space multiply of the cuFFT comparison pipeline (the "custom CUDA kernel for
//                  intermediate operations" of PAPER.md:115), so that the comparison is against a tight cuFFT
//                  pipeline and not against eager tensor arithmetic.
// They give SURVEY.md 8(d) "Which roofline" its measured ALU / shared-memory denominators on the box the bench runs on.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

constexpr int kChains = 8;

__global__ void __launch_bounds__(256) k_fp64(double* out, int iters, double a, double b)
{
    double v[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) v[c] = (double)(threadIdx.x + c) * 1e-3;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) v[c] = fma(v[c], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < kChains; ++c) s += v[c];
    if (s == 12345.678) out[blockIdx.x * blockDim.x + threadIdx.x] = s;     // keeps the chains alive, never true
}

__global__ void __launch_bounds__(256) k_lds(double* out, int iters)
{
    __shared__ double2 buf[2048];                    // 32 KB
    for (int i = threadIdx.x; i < 2048; i += 256) buf[i] = make_double2((double)i, 1.0);
    __syncthreads();
    double2 acc = make_double2(0.0, 0.0);
    int idx = threadIdx.x;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const double2 v = buf[(idx + u * 256) & 2047];     // a warp reads 512 contiguous bytes: conflict free
            acc.x += v.x;
            acc.y += v.y;
        }
        idx = (idx + 8) & 2047;
    }
    if (acc.x + acc.y == -1.0) out[blockIdx.x * blockDim.x + threadIdx.x] = acc.x;
}

__global__ void __launch_bounds__(256) k_l2(const double2* __restrict__ in, double* out, int64_t n, int reps)
{
    double2 acc = make_double2(0.0, 0.0);
    for (int r = 0; r < reps; ++r)
        for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (int64_t)gridDim.x * 256) {
            double2 v;
            asm volatile("ld.global.cg.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(in + i));
            acc.x += v.x;
            acc.y += v.y;
        }
    if (acc.x + acc.y == -1.0) out[blockIdx.x * 256 + threadIdx.x] = acc.x;
}

// E~_i = sum_j K_ij P~_j, K real symmetric (xx yy zz xy xz yz); P, E complex [B][3][n]; K [6][n]
template <typename T>
__global__ void __launch_bounds__(256) k_kmul(const T* __restrict__ P, const T* __restrict__ K, T* __restrict__ E, int64_t n,
                                              int batch)
{
    for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += (int64_t)gridDim.x * 256) {
        const T kxx = K[i], kyy = K[n + i], kzz = K[2 * n + i], kxy = K[3 * n + i], kxz = K[4 * n + i], kyz = K[5 * n + i];
        for (int b = 0; b < batch; ++b) {
            const T* p = P + (int64_t)b * 6 * n;
            T* e = E + (int64_t)b * 6 * n;
            const T pxr = p[2 * i], pxi = p[2 * i + 1], pyr = p[2 * (n + i)], pyi = p[2 * (n + i) + 1];
            const T pzr = p[2 * (2 * n + i)], pzi = p[2 * (2 * n + i) + 1];
            e[2 * i] = kxx * pxr + kxy * pyr + kxz * pzr;
            e[2 * i + 1] = kxx * pxi + kxy * pyi + kxz * pzi;
            e[2 * (n + i)] = kxy * pxr + kyy * pyr + kyz * pzr;
            e[2 * (n + i) + 1] = kxy * pxi + kyy * pyi + kyz * pzi;
            e[2 * (2 * n + i)] = kxz * pxr + kyz * pyr + kzz * pzr;
            e[2 * (2 * n + i) + 1] = kxz * pxi + kyz * pyi + kzz * pzi;
        }
    }
}

// warps 0-3 of a block run the DFMA chains, warps 4-7 the shared-memory loads: mode 1 = fp64 only, 2 = loads only,
// 3 = both at once.  If the two units are independent, mode 3 takes max(mode 1, mode 2); if they share a resource, the sum.
__global__ void __launch_bounds__(256) k_mix(double* out, int iters, double a, double b, int mode)
{
    __shared__ double2 buf[2048];
    for (int i = threadIdx.x; i < 2048; i += 256) buf[i] = make_double2((double)i, 1.0);
    __syncthreads();
    const int warp = threadIdx.x >> 5;
    double s = 0.0;
    if (warp < 4) {
        if (mode & 1) {
            double v[kChains];
#pragma unroll
            for (int c = 0; c < kChains; ++c) v[c] = (double)(threadIdx.x + c) * 1e-3;
            for (int i = 0; i < iters; ++i) {
#pragma unroll
                for (int u = 0; u < 4; ++u) {
#pragma unroll
                    for (int c = 0; c < kChains; ++c) v[c] = fma(v[c], a, b);
                }
            }
#pragma unroll
            for (int c = 0; c < kChains; ++c) s += v[c];
        }
    } else if (mode & 2) {
        double2 acc = make_double2(0.0, 0.0);
        int idx = threadIdx.x;
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const double2 v = buf[(idx + u * 256) & 2047];
                acc.x += v.x;      // two DADD per load: small against the 4 wavefronts of the load
                acc.y += v.y;
            }
            idx = (idx + 8) & 2047;
        }
        s = acc.x + acc.y;
    }
    if (s == 12345.678) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

struct Timer {
    cudaEvent_t e0, e1;
    Timer() { cudaEventCreate(&e0); cudaEventCreate(&e1); }
    ~Timer() { cudaEventDestroy(e0); cudaEventDestroy(e1); }
    void start(cudaStream_t st) { cudaEventRecord(e0, st); }
    float stop(cudaStream_t st)
    {
        float ms = 0.f;
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        cudaEventElapsedTime(&ms, e0, e1);
        return ms;
    }
};

int sm_count()
{
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    return sms;
}

}  // namespace

// out_inst_per_s: fp64 WARP instructions per second of the whole device (one DFMA = 2 flops x 32 lanes).
// scratch: device memory of at least 8 * 256 * blocks doubles (never written).  Returns 0 on success.
extern "C" int fe_peak_fp64(void* scratch, int blocks_per_sm, int iters, double* out_inst_per_s, void* stream)
{
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int grid = sm_count() * blocks_per_sm;
    Timer t;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        t.start(st);
        k_fp64<<<grid, 256, 0, st>>>(static_cast<double*>(scratch), iters, 0.999999, 1e-7);
        const float ms = t.stop(st);
        if (cudaGetLastError() != cudaSuccess || ms <= 0.f) return 1;
        const double inst = (double)grid * 8 /* warps */ * iters * 4.0 * kChains;
        const double r = inst / (ms * 1e-3);
        if (rep > 0 && r > best) best = r;
    }
    *out_inst_per_s = best;
    return 0;
}

// out_ms[3]: time of k_mix in mode 1 (fp64 on half the warps), 2 (shared-memory loads on the other half), 3 (both)
extern "C" int fe_peak_mix(void* scratch, int iters, double* out_ms, void* stream)
{
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int grid = sm_count();
    Timer t;
    for (int mode = 1; mode <= 3; ++mode) {
        float best = 1e30f;
        for (int rep = 0; rep < 3; ++rep) {
            t.start(st);
            k_mix<<<grid, 256, 0, st>>>(static_cast<double*>(scratch), iters, 0.999999, 1e-7, mode);
            const float ms = t.stop(st);
            if (cudaGetLastError() != cudaSuccess || ms <= 0.f) return 1;
            if (rep > 0 && ms < best) best = ms;
        }
        out_ms[mode - 1] = best;
    }
    return 0;
}

// out_bytes_per_s: shared-memory read bandwidth of the whole device
extern "C" int fe_peak_lds(void* scratch, int blocks_per_sm, int iters, double* out_bytes_per_s, void* stream)
{
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int grid = sm_count() * blocks_per_sm;
    Timer t;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        t.start(st);
        k_lds<<<grid, 256, 0, st>>>(static_cast<double*>(scratch), iters);
        const float ms = t.stop(st);
        if (cudaGetLastError() != cudaSuccess || ms <= 0.f) return 1;
        const double bytes = (double)grid * 256 * iters * 8.0 * 16.0;
        const double r = bytes / (ms * 1e-3);
        if (rep > 0 && r > best) best = r;
    }
    *out_bytes_per_s = best;
    return 0;
}

// out_bytes_per_s: read bandwidth of `bytes` (a multiple of 16) of device memory read `reps` times by one kernel;
// with bytes well below the L2 capacity this is the L2 read bandwidth
extern "C" int fe_peak_l2(const void* buf, void* scratch, int64_t bytes, int reps, double* out_bytes_per_s, void* stream)
{
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int grid = sm_count() * 8;
    Timer t;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        t.start(st);
        k_l2<<<grid, 256, 0, st>>>(static_cast<const double2*>(buf), static_cast<double*>(scratch), bytes / 16, reps);
        const float ms = t.stop(st);
        if (cudaGetLastError() != cudaSuccess || ms <= 0.f) return 1;
        const double r = (double)bytes * reps / (ms * 1e-3);
        if (rep > 0 && r > best) best = r;
    }
    *out_bytes_per_s = best;
    return 0;
}

// P, E: complex spectra [batch][3][n] (interleaved re, im), K: real [6][n]; f32 != 0: float, else double
extern "C" int fe_bench_kmul(const void* P, const void* K, void* E, int64_t n, int batch, int f32, void* stream)
{
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int grid = sm_count() * 8;
    if (f32) k_kmul<float><<<grid, 256, 0, st>>>((const float*)P, (const float*)K, (float*)E, n, batch);
    else k_kmul<double><<<grid, 256, 0, st>>>((const double*)P, (const double*)K, (double*)E, n, batch);
    return cudaGetLastError() == cudaSuccess ? 0 : 1;
}
