// fe_fft2_axis.cu -- size-specialised strided pass along y:
// forward reads n_keep rows (the rest of the padded axis is zero) and writes M rows, inverse reads M rows and
// writes n_keep rows.  A tile is M rows x 128 bytes of consecutive kx; the transform runs in registers with
// one shared-memory exchange (fe_fft2.cuh).
#include "fe_fft2.cuh"
#include <stdlib.h>

namespace fe {
namespace v2 {

// A tile is M rows of LANES consecutive complex elements.  Its first element sits at
// blockIdx.x * s0 + blockIdx.y * s1 + blockIdx.z * sb, its rows are sa apart (all in complex elements), so the
// same kernels serve the row-major spectra and the tiled layouts of fe_api.cu.
struct Axis2Args {
    const void* tw;
    int64_t in_sa, in_s0, in_s1, in_sb, out_sa, out_s0, out_s1, out_sb;
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
    const cx<T>* ib = in + (int64_t)blockIdx.z * a.in_sb + (int64_t)blockIdx.y * a.in_s1 + (int64_t)blockIdx.x * a.in_s0 + lane;
    cx<T>* ob = out + (int64_t)blockIdx.z * a.out_sb + (int64_t)blockIdx.y * a.out_s1 + (int64_t)blockIdx.x * a.out_s0 + lane;

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

// ------------------------------------------------------------------------------------------------
// Three-level variant for the long axes (M = 256, 512): M = RA * RB * RC,
//   n = n3 + RC n2 + RC RB n1,   k = k1 + RA k2 + RA RB k3,
//   A: RA-point over n1, twiddle w_M^((n3 + RC n2) k1);  B: RB-point over n2 (in place), twiddle w_M^(RA n3 k2);
//   C: RC-point over n3.
// A thread holds at most 8 points, so a 256-thread block needs ~80 registers per thread and three blocks share
// an SM (24 warps instead of 12): the passes are latency bound and trade a second shared-memory exchange for
// twice the warps in flight.
// ------------------------------------------------------------------------------------------------
template <int M> struct Fact3;
template <> struct Fact3<256> { static constexpr int RA = 8, RB = 8, RC = 4; };
template <> struct Fact3<512> { static constexpr int RA = 8, RB = 8, RC = 8; };

template <typename T, int M, int DIR, bool PRUNE>
__global__ void __launch_bounds__(256, 3)
k3_axis(const cx<T>* __restrict__ in, cx<T>* __restrict__ out, Axis2Args a)
{
    constexpr int RA = Fact3<M>::RA, RB = Fact3<M>::RB, RC = Fact3<M>::RC;
    constexpr int LANES = 128 / (int)sizeof(cx<T>);
    constexpr int TPP = 256 / LANES;                          // threads per pencil
    constexpr int NTA = RB * RC, NTB = RA * RC, NTC = RA * RB;  // tasks per pencil and level
    static_assert(NTA % TPP == 0 && NTB % TPP == 0 && NTC % TPP == 0, "tasks must divide evenly");
    cx<T>* tw = reinterpret_cast<cx<T>*>(fe2_smem);
    cx<T>* buf = tw + M;
    const int lane = threadIdx.x % LANES, tp = threadIdx.x / LANES;
    const cx<T>* ib = in + (int64_t)blockIdx.z * a.in_sb + (int64_t)blockIdx.y * a.in_s1 + (int64_t)blockIdx.x * a.in_s0 + lane;
    cx<T>* ob = out + (int64_t)blockIdx.z * a.out_sb + (int64_t)blockIdx.y * a.out_s1 + (int64_t)blockIdx.x * a.out_s0 + lane;
    constexpr bool PIN = PRUNE && DIR < 0, POUT = PRUNE && DIR > 0;
    constexpr int NLOAD = PIN ? RA / 2 : RA;

    // ---- level A: task j = n3 + RC n2 holds x[j + RB RC n1]
    cx<T> va[NTA / TPP][RA];
#pragma unroll
    for (int it = 0; it < NTA / TPP; ++it) {
        const int j = tp + it * TPP;
        static_for<NLOAD>([&](auto ic) {
            constexpr int n1 = decltype(ic)::value;
            va[it][n1] = ib[(int64_t)(j + RB * RC * n1) * a.in_sa];
        });
    }
    load_twiddles<T, M>(tw, static_cast<const cx<T>*>(a.tw), threadIdx.x, 256);
    __syncthreads();
#pragma unroll
    for (int it = 0; it < NTA / TPP; ++it) {
        const int j = tp + it * TPP;
        Dif<T, DIR, RA, 0, PIN>::run(va[it]);
        static_for<RA>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            constexpr int k1 = brev<RA>(p);
            cx<T> val = va[it][p];
            if constexpr (k1 != 0) val = cmuld<T, DIR>(val, tw[j * k1]);
            buf[(k1 * RB * RC + j) * LANES + lane] = val;      // (k1, n2, n3) at (k1 RB + n2) RC + n3
        });
    }
    __syncthreads();
    // ---- level B (in place): task (k1, n3)
#pragma unroll
    for (int it = 0; it < NTB / TPP; ++it) {
        const int tb = tp + it * TPP, n3 = tb % RC, k1 = tb / RC;
        cx<T> u[RB];
        cx<T>* col = buf + (k1 * RB * RC + n3) * LANES + lane;
        static_for<RB>([&](auto nc) { u[decltype(nc)::value] = col[decltype(nc)::value * RC * LANES]; });
        Dif<T, DIR, RB>::run(u);
        static_for<RB>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            constexpr int k2 = brev<RB>(p);
            cx<T> val = u[p];
            if constexpr (k2 != 0) val = cmuld<T, DIR>(val, tw[RA * n3 * k2]);
            col[k2 * RC * LANES] = val;
        });
    }
    __syncthreads();
    // ---- level C: task (k1, k2), rows k1 + RA k2 + RA RB k3
#pragma unroll
    for (int it = 0; it < NTC / TPP; ++it) {
        const int tc = tp + it * TPP, k1 = tc % RA, k2 = tc / RA;
        cx<T> u[RC];
        const cx<T>* src = buf + ((k1 * RB + k2) * RC) * LANES + lane;
        static_for<RC>([&](auto nc) { u[decltype(nc)::value] = src[decltype(nc)::value * LANES]; });
        Dif<T, DIR, RC>::run(u);
        static_for<RC>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            constexpr int k3 = brev<RC>(p);
            if constexpr (!POUT || k3 < RC / 2) ob[(int64_t)(tc + RA * RB * k3) * a.out_sa] = u[p];
        });
    }
}

template <typename T, int M, int DIR, bool PRUNE>
static cudaError_t launch_one3(const void* in, void* out, const Axis2Args& a, dim3 grid, cudaStream_t st)
{
    constexpr int LANES = 128 / (int)sizeof(cx<T>);
    constexpr size_t smem = (size_t)(M + M * LANES) * sizeof(cx<T>);
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(k3_axis<T, M, DIR, PRUNE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    k3_axis<T, M, DIR, PRUNE><<<grid, 256, smem, st>>>(static_cast<const cx<T>*>(in), static_cast<cx<T>*>(out), a);
    return cudaGetLastError();
}

template <typename T, int M>
static cudaError_t launch_m3(int dir, bool prune, const void* in, void* out, const Axis2Args& a, dim3 grid,
                             cudaStream_t st)
{
    if (dir < 0) return prune ? launch_one3<T, M, -1, true>(in, out, a, grid, st)
                              : launch_one3<T, M, -1, false>(in, out, a, grid, st);
    return prune ? launch_one3<T, M, +1, true>(in, out, a, grid, st) : launch_one3<T, M, +1, false>(in, out, a, grid, st);
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

// Strided pass along one axis (axis = 1 or 2 picks the plan).  Grid (n0, n1, batch); see Axis2Args for the strides.
// n_keep = M (periodic axis) or M / 2 (zero-padded axis: forward reads, inverse writes only the first half).
template <typename T>
cudaError_t launch_axis2(const FftCtx& c, int axis, int dir, const void* in, void* out, int n_keep, int n0, int n1,
                         int batch, int64_t in_sa, int64_t in_s0, int64_t in_s1, int64_t in_sb, int64_t out_sa,
                         int64_t out_s0, int64_t out_s1, int64_t out_sb, cudaStream_t st)
{
    const int M = c.plan[axis].M;
    v2::Axis2Args a{c.tw, in_sa, in_s0, in_s1, in_sb, out_sa, out_s0, out_s1, out_sb};
    dim3 grid(n0, n1, batch);
    const bool prune = 2 * n_keep == M;
    if (!prune && n_keep != M) return cudaErrorInvalidValue;
    static const bool three_level = getenv("FE_B200_Y3") && getenv("FE_B200_Y3")[0] == '1';   // tuning aid
    if (three_level) {
        if (M == 256) return v2::launch_m3<T, 256>(dir, prune, in, out, a, grid, st);
        if (M == 512) return v2::launch_m3<T, 512>(dir, prune, in, out, a, grid, st);
    }
    switch (M) {
        case 64: return v2::launch_m<T, 64>(dir, prune, in, out, a, grid, st);
        case 128: return v2::launch_m<T, 128>(dir, prune, in, out, a, grid, st);
        case 256: return v2::launch_m<T, 256>(dir, prune, in, out, a, grid, st);
        case 512: return v2::launch_m<T, 512>(dir, prune, in, out, a, grid, st);
        default: return cudaErrorInvalidValue;
    }
}

template cudaError_t launch_axis2<double>(const FftCtx&, int, int, const void*, void*, int, int, int, int, int64_t,
                                          int64_t, int64_t, int64_t, int64_t, int64_t, int64_t, int64_t, cudaStream_t);
template cudaError_t launch_axis2<float>(const FftCtx&, int, int, const void*, void*, int, int, int, int, int64_t,
                                         int64_t, int64_t, int64_t, int64_t, int64_t, int64_t, int64_t, cudaStream_t);

}  // namespace fe
