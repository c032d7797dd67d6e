// fe_fft2_axis.cu -- size-specialised strided pass along y:
// forward reads n_keep rows (the rest of the padded axis is zero) and writes M rows, inverse reads M rows and
// writes n_keep rows.  A tile is M rows x 128 bytes of consecutive kx; the transform runs in registers with
// one shared-memory exchange (fe_fft2.cuh).
#include "fe_fft2.cuh"

namespace fe {
namespace v2 {

struct Axis2Args {
    const void* tw;
    int64_t in_sa, in_so, in_sb, out_sa, out_so, out_sb;
};

template <typename T, int M, int DIR, bool PRUNE>
__global__ void __launch_bounds__((128 / (int)sizeof(cx<T>)) * Fact<M>::R2)
k2_axis(const cx<T>* __restrict__ in, cx<T>* __restrict__ out, Axis2Args a)
{
    constexpr int R1 = Fact<M>::R1, R2 = Fact<M>::R2;
    constexpr int LANES = 128 / (int)sizeof(cx<T>);
    constexpr int TPP = R2;                     // threads per pencil
    constexpr int NT3 = R1 / TPP;               // step-3 tasks per thread
    cx<T>* tw = reinterpret_cast<cx<T>*>(fe2_smem);
    cx<T>* buf = tw + M;
    const int lane = threadIdx.x % LANES, tp = threadIdx.x / LANES;
    const int kx0 = blockIdx.x * LANES;
    const cx<T>* ib = in + (int64_t)blockIdx.z * a.in_sb + (int64_t)blockIdx.y * a.in_so + kx0 + lane;
    cx<T>* ob = out + (int64_t)blockIdx.z * a.out_sb + (int64_t)blockIdx.y * a.out_so + kx0 + lane;

    // step 1: thread n2 = tp holds x[n2 + R2 n1]
    cx<T> v[R1];
    constexpr bool PIN = PRUNE && DIR < 0;      // zero-padded input (forward)
    constexpr int NLOAD = PIN ? R1 / 2 : R1;
    static_for<NLOAD>([&](auto ic) {
        constexpr int n1 = decltype(ic)::value;
        const int row = tp + R2 * n1;
        v[n1] = ib[(int64_t)row * a.in_sa];
    });
    load_twiddles<T, M>(tw, static_cast<const cx<T>*>(a.tw), threadIdx.x, LANES * TPP);
    __syncthreads();
    Dif<T, DIR, R1, 0, PIN>::run(v);
    static_for<R1>([&](auto pc) {
        constexpr int p = decltype(pc)::value;
        constexpr int k1 = brev<R1>(p);
        cx<T> val = v[p];
        if constexpr (k1 != 0) val = cmuld<T, DIR>(val, tw[tp * k1]);
        buf[(k1 * R2 + tp) * LANES + lane] = val;
    });
    __syncthreads();
    // step 3: thread k1 = tp (+ TPP ...) runs the R2-point transform over n2
    constexpr bool POUT = PRUNE && DIR > 0;     // only the first half of the outputs is kept (inverse)
#pragma unroll
    for (int it = 0; it < NT3; ++it) {
        const int k1 = tp + it * TPP;
        cx<T> u[R2];
        static_for<R2>([&](auto nc) {
            constexpr int n2 = decltype(nc)::value;
            u[n2] = buf[(k1 * R2 + n2) * LANES + lane];
        });
        Dif<T, DIR, R2>::run(u);
        static_for<R2>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            constexpr int k2 = brev<R2>(p);
            if constexpr (!POUT || k2 < R2 / 2) {
                const int row = k1 + R1 * k2;
                ob[(int64_t)row * a.out_sa] = u[p];
            }
        });
    }
}

template <typename T, int M, int DIR, bool PRUNE>
static cudaError_t launch_one(const void* in, void* out, const Axis2Args& a, dim3 grid, cudaStream_t st)
{
    constexpr int LANES = 128 / (int)sizeof(cx<T>);
    constexpr int threads = LANES * Fact<M>::R2;
    constexpr size_t smem = (size_t)(M + M * LANES) * sizeof(cx<T>);
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(k2_axis<T, M, DIR, PRUNE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    k2_axis<T, M, DIR, PRUNE><<<grid, threads, smem, st>>>(static_cast<const cx<T>*>(in), static_cast<cx<T>*>(out), a);
    return cudaGetLastError();
}

template <typename T, int M>
static cudaError_t launch_m(int dir, bool prune, const void* in, void* out, const Axis2Args& a, dim3 grid,
                            cudaStream_t st)
{
    if (dir < 0) return prune ? launch_one<T, M, -1, true>(in, out, a, grid, st)
                              : launch_one<T, M, -1, false>(in, out, a, grid, st);
    return prune ? launch_one<T, M, +1, true>(in, out, a, grid, st) : launch_one<T, M, +1, false>(in, out, a, grid, st);
}

}  // namespace v2

bool axis2_supported(int M) { return M == 64 || M == 128 || M == 256 || M == 512; }

// same contract as launch_axis (fe_fft.cu), natural frequency order on the spectrum side
template <typename T>
cudaError_t launch_axis2(const FftCtx& c, int axis, int dir, const void* in, void* out, int n_keep, int pitch_used,
                         int outer, int batch, int64_t in_sa, int64_t in_so, int64_t in_sb, int64_t out_sa,
                         int64_t out_so, int64_t out_sb, cudaStream_t st)
{
    const int M = c.plan[axis].M;
    constexpr int LANES = 128 / (int)sizeof(v2::cx<T>);
    v2::Axis2Args a{c.tw, in_sa, in_so, in_sb, out_sa, out_so, out_sb};
    dim3 grid(pitch_used / LANES, outer, batch);
    const bool prune = 2 * n_keep == M;
    if (!prune && n_keep != M) return cudaErrorInvalidValue;
    switch (M) {
        case 64: return v2::launch_m<T, 64>(dir, prune, in, out, a, grid, st);
        case 128: return v2::launch_m<T, 128>(dir, prune, in, out, a, grid, st);
        case 256: return v2::launch_m<T, 256>(dir, prune, in, out, a, grid, st);
        case 512: return v2::launch_m<T, 512>(dir, prune, in, out, a, grid, st);
        default: return cudaErrorInvalidValue;
    }
}

template cudaError_t launch_axis2<double>(const FftCtx&, int, int, const void*, void*, int, int, int, int, int64_t,
                                          int64_t, int64_t, int64_t, int64_t, int64_t, cudaStream_t);
template cudaError_t launch_axis2<float>(const FftCtx&, int, int, const void*, void*, int, int, int, int, int64_t,
                                         int64_t, int64_t, int64_t, int64_t, int64_t, cudaStream_t);

}  // namespace fe
