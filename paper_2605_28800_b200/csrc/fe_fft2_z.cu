// fe_fft2_z.cu -- size-specialised fused z pass (Eq. 5-6 in k-space):
// forward z transform of the three components, E~_i = -escale * sum_j K~_ij P~_j, inverse z transform, in place
// on S[b][3][nz][My][pitch].  K~ is real and symmetric, stored for kz <= Mz/2, ky <= My/2; the odd components
// change sign under ky -> -ky (xy, yz) and kz -> -kz (xz, yz).
//
// One thread holds the spectrum of all three components at the R2 frequencies kz = k1 + R1 k2 in registers, so
// the multiply and the first stage of the inverse transform need no shared memory:
//   forward   x[n2 + R2 n1] -> (R1-point over n1) -> twiddle -> exchange -> (R2-point over n2) -> X[k1 + R1 k2]
//   inverse   X[k1 + R1 k2] -> (R2-point over k2) -> twiddle -> exchange -> (R1-point over k1) -> x[n1 R2 + n2]
// The thread that loaded rows n2 + R2 n1 stores exactly those rows again.
#include "fe_fft2.cuh"

namespace fe {
namespace v2 {

struct Z2Args {
    const void* tw;
    const DevMember* members;
    int My, pitch;
    int nz;
};

template <typename T, int M, bool PRUNE>
__global__ void __launch_bounds__((128 / (int)sizeof(cx<T>)) * Fact<M>::R1, 2)
k2_zmul(cx<T>* __restrict__ S, const T* __restrict__ Kt, Z2Args a)
{
    constexpr int R1 = Fact<M>::R1, R2 = Fact<M>::R2;
    constexpr int LANES = 128 / (int)sizeof(cx<T>);
    constexpr int TPP = R1;                                 // threads per pencil (one step-3 task each)
    constexpr int NT1 = (3 * R2 + TPP - 1) / TPP;           // step-1 tasks (component, n2) per thread
    constexpr int TILE = M * LANES;
    constexpr int NLOAD = PRUNE ? R1 / 2 : R1;
    cx<T>* tw = reinterpret_cast<cx<T>*>(fe2_smem);
    cx<T>* buf = tw + M;
    const int lane = threadIdx.x % LANES, tp = threadIdx.x / LANES;
    const int kx0 = blockIdx.x * LANES, b = blockIdx.z;
    // mirror pairs (ky, My - ky) are adjacent in launch order so that the second read of a K~ plane hits L2
    const int yy = blockIdx.y;
    const int ky = yy == 0 ? 0 : ((yy & 1) ? (yy + 1) >> 1 : a.My - (yy >> 1));
    const int64_t sa = (int64_t)a.My * a.pitch, cs = (int64_t)a.nz * sa;
    cx<T>* base = S + (int64_t)b * 3 * cs + (int64_t)ky * a.pitch + kx0 + lane;

    // ---- forward step 1: tasks (c, n2)
    cx<T> v[NT1][NLOAD];
#pragma unroll
    for (int it = 0; it < NT1; ++it) {
        const int task = tp + it * TPP;
        if ((3 * R2) % TPP == 0 || task < 3 * R2) {
            const int c = task / R2, n2 = task % R2;
            const cx<T>* src = base + c * cs + (int64_t)n2 * sa;
            static_for<NLOAD>([&](auto ic) {
                constexpr int n1 = decltype(ic)::value;
                v[it][n1] = src[(int64_t)(R2 * n1) * sa];
            });
        }
    }
    load_twiddles<T, M>(tw, static_cast<const cx<T>*>(a.tw), threadIdx.x, LANES * TPP);
    __syncthreads();
#pragma unroll
    for (int it = 0; it < NT1; ++it) {
        const int task = tp + it * TPP;
        if ((3 * R2) % TPP == 0 || task < 3 * R2) {
            const int c = task / R2, n2 = task % R2;
            cx<T> w[R1];
            static_for<NLOAD>([&](auto ic) { w[decltype(ic)::value] = v[it][decltype(ic)::value]; });
            Dif<T, -1, R1, 0, PRUNE>::run(w);
            cx<T>* dst = buf + c * TILE + n2 * LANES + lane;
            static_for<R1>([&](auto pc) {
                constexpr int p = decltype(pc)::value;
                constexpr int k1 = brev<R1>(p);
                cx<T> val = w[p];
                if constexpr (k1 != 0) val = cmul(val, tw[n2 * k1]);
                dst[k1 * R2 * LANES] = val;
            });
        }
    }
    __syncthreads();
    // ---- forward step 3 for thread k1 = tp: u[c][p] = P~_c[k1 + R1 brev(p)]
    const int k1 = tp;
    cx<T> u[3][R2];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const cx<T>* src = buf + c * TILE + k1 * R2 * LANES + lane;
        static_for<R2>([&](auto nc) { u[c][decltype(nc)::value] = src[decltype(nc)::value * LANES]; });
        Dif<T, -1, R2>::run(u[c]);
    }
    __syncthreads();     // every thread has read its forward data: the buffers may be overwritten
    // ---- multiply
    {
        const int Hy = a.My / 2 + 1, Hz = M / 2 + 1;
        const int kym = ky <= a.My / 2 ? ky : a.My - ky;
        const T esc = (T)(-a.members[b].escale);
        const T sy = ky > a.My / 2 ? -esc : esc;
        const int64_t kcs = (int64_t)Hz * Hy * a.pitch;
        const T* kb = Kt + (int64_t)kym * a.pitch + kx0 + lane;
        static_for<R2>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            constexpr int k2 = brev<R2>(p);
            const int kz = k1 + R1 * k2;
            const int kzm = kz <= M / 2 ? kz : M - kz;
            const T* kp = kb + (int64_t)kzm * Hy * a.pitch;
            const T sz = kz > M / 2 ? (T)-1 : (T)1;
            const T Kxx = esc * __ldg(kp), Kyy = esc * __ldg(kp + kcs), Kzz = esc * __ldg(kp + 2 * kcs);
            const T Kxy = sy * __ldg(kp + 3 * kcs), Kxz = esc * sz * __ldg(kp + 4 * kcs);
            const T Kyz = sy * sz * __ldg(kp + 5 * kcs);
            const cx<T> Px = u[0][p], Py = u[1][p], Pz = u[2][p];
            u[0][p] = {Kxx * Px.x + Kxy * Py.x + Kxz * Pz.x, Kxx * Px.y + Kxy * Py.y + Kxz * Pz.y};
            u[1][p] = {Kxy * Px.x + Kyy * Py.x + Kyz * Pz.x, Kxy * Px.y + Kyy * Py.y + Kyz * Pz.y};
            u[2][p] = {Kxz * Px.x + Kyz * Py.x + Kzz * Pz.x, Kxz * Px.y + Kyz * Py.y + Kzz * Pz.y};
        });
    }
    // ---- inverse step 1: R2-point over k2 (bit-reversed in, natural n2 out), twiddle, exchange
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        Dit<T, +1, R2>::run(u[c]);
        cx<T>* dst = buf + c * TILE + k1 * LANES + lane;
        static_for<R2>([&](auto nc) {
            constexpr int n2 = decltype(nc)::value;
            cx<T> val = u[c][n2];
            if constexpr (n2 != 0) val = cmulc(val, tw[n2 * k1]);
            dst[n2 * R1 * LANES] = val;
        });
    }
    __syncthreads();
    // ---- inverse step 2: tasks (c, n2): R1-point over k1, rows n1 R2 + n2 (n1 < R1/2 when pruned) stored
#pragma unroll
    for (int it = 0; it < NT1; ++it) {
        const int task = tp + it * TPP;
        if ((3 * R2) % TPP == 0 || task < 3 * R2) {
            const int c = task / R2, n2 = task % R2;
            cx<T> w[R1];
            const cx<T>* src = buf + c * TILE + n2 * R1 * LANES + lane;
            static_for<R1>([&](auto kc) { w[decltype(kc)::value] = src[decltype(kc)::value * LANES]; });
            Dif<T, +1, R1>::run(w);
            cx<T>* out = base + c * cs + (int64_t)n2 * sa;
            static_for<R1>([&](auto pc) {
                constexpr int p = decltype(pc)::value;
                constexpr int n1 = brev<R1>(p);
                if constexpr (!PRUNE || n1 < R1 / 2) out[(int64_t)(R2 * n1) * sa] = w[p];
            });
        }
    }
}

template <typename T, int M, bool PRUNE>
static cudaError_t launch_one(void* S, const T* Kt, const Z2Args& a, dim3 grid, cudaStream_t st)
{
    constexpr int LANES = 128 / (int)sizeof(cx<T>);
    constexpr int threads = LANES * Fact<M>::R1;
    constexpr size_t smem = (size_t)(M + 3 * M * LANES) * sizeof(cx<T>);
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(k2_zmul<T, M, PRUNE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    k2_zmul<T, M, PRUNE><<<grid, threads, smem, st>>>(static_cast<cx<T>*>(S), Kt, a);
    return cudaGetLastError();
}

}  // namespace v2

bool zmul2_supported(int M) { return M == 64 || M == 128 || M == 256; }

// same contract as launch_zmul (fe_fft.cu)
template <typename T>
cudaError_t launch_zmul2(const FftCtx& c, void* S, const T* Kt, const DevMember* members, int nz, int My, int pitch,
                         int batch, cudaStream_t st)
{
    const int M = c.plan[2].M;
    constexpr int LANES = 128 / (int)sizeof(v2::cx<T>);
    v2::Z2Args a{c.tw, members, My, pitch, nz};
    dim3 grid(pitch / LANES, My, batch);
    const bool prune = 2 * nz == M;
    if (!prune && nz != M) return cudaErrorInvalidValue;
    switch (M) {
        case 64: return prune ? v2::launch_one<T, 64, true>(S, Kt, a, grid, st) : v2::launch_one<T, 64, false>(S, Kt, a, grid, st);
        case 128: return prune ? v2::launch_one<T, 128, true>(S, Kt, a, grid, st) : v2::launch_one<T, 128, false>(S, Kt, a, grid, st);
        case 256: return prune ? v2::launch_one<T, 256, true>(S, Kt, a, grid, st) : v2::launch_one<T, 256, false>(S, Kt, a, grid, st);
        default: return cudaErrorInvalidValue;
    }
}

template cudaError_t launch_zmul2<double>(const FftCtx&, void*, const double*, const DevMember*, int, int, int, int,
                                          cudaStream_t);
template cudaError_t launch_zmul2<float>(const FftCtx&, void*, const float*, const DevMember*, int, int, int, int,
                                         cudaStream_t);

}  // namespace fe
