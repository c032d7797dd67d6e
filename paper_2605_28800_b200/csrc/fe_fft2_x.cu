// fe_fft2_x.cu -- size-specialised x passes: real rows of n_x
// values (zero-padded to m_x = 2 M when the axis is open) <-> half spectra X[0..M].
// The real transform of length 2 M runs as a complex transform of length M on z[j] = x[2j] + i x[2j+1]:
//   forward  Z = FFT_M(z);  X[k] = (Z[k] + conj Z[M-k])/2 - (i/2) w_2M^k (Z[k] - conj Z[M-k])
//   inverse  Z[k] = (X[k] + conj X[M-k])/2 + (i/2) conj(w_2M^k) (X[k] - conj X[M-k]);  z = M * IFFT_M(Z)
// (the inverse is unnormalised; 1/(M m_y m_z) is folded into the tensor spectrum at precompute).
// Each row is handled by R2 threads with the register two-level transform of fe_fft2.cuh.
#include "fe_fft2.cuh"

namespace fe {
namespace v2 {

// Real row r starts at r * real_rs.  Spectrum element k of row r sits at
// (r / ny) * s_plane + (r % ny) * s_row + (k >> lg) * s_g + (k & (2^lg - 1))   (complex elements; 2^lg = kx per group),
// which covers the row-major spectra (s_g = 2^lg) and the tiled layout of fe_api.cu.
struct X2Args {
    const void* tw;
    int64_t nrows;
    int64_t real_rs;
    int ny, lg;
    int64_t s_plane, s_row, s_g;
    int nc;         // valid complex pairs (x[2j], x[2j+1]) per real row: n_x / 2 (<= M/2 on a zero-padded axis, M otherwise)
};
__device__ __forceinline__ int64_t spec_off(const X2Args& a, int k) { return (int64_t)(k >> a.lg) * a.s_g + (k & ((1 << a.lg) - 1)); }
__device__ __forceinline__ int64_t spec_row(const X2Args& a, int64_t row) { return (row / a.ny) * a.s_plane + (row % a.ny) * a.s_row; }

template <int M> struct XCfg {
    static constexpr int R1 = Fact<M>::R1, R2 = Fact<M>::R2;
    static constexpr int TPP = R2;
    static constexpr int ROWS = 256 / TPP;            // rows per block (256 threads)
    static constexpr int XPITCH = R1 * (R2 + 1);      // padded exchange layout idx(k1, n2) = k1 (R2+1) + n2
    static constexpr int RPITCH = XPITCH > M + 1 ? XPITCH : M + 1;
};

template <typename T, int M, bool PRUNE>
__global__ void __launch_bounds__(256, M >= 512 ? 1 : 2) k2_xfwd(const T* __restrict__ in, cx<T>* __restrict__ out, X2Args a)
{
    using C = XCfg<M>;
    constexpr int R1 = C::R1, R2 = C::R2, TPP = C::TPP, NT3 = R1 / TPP;
    cx<T>* tw = reinterpret_cast<cx<T>*>(fe2_smem);   // w_M^e
    cx<T>* tws = tw + M;                              // w_2M^k, k < M
    cx<T>* buf = tws + M;
    const int tp = threadIdx.x % TPP, rl = threadIdx.x / TPP;
    cx<T>* rb = buf + rl * C::RPITCH;
    constexpr int NLOAD = PRUNE ? R1 / 2 : R1;
    // persistent: a block walks over groups of ROWS rows; the real input of the next group is fetched into registers
    // before the current group is transformed, so the global-load latency hides behind a whole group of work
    const int64_t ngroups = (a.nrows + C::ROWS - 1) / C::ROWS;
    auto fetch = [&](int64_t grp, cx<T>* dst) {
        const int64_t row = grp * C::ROWS + rl;
        if (grp < ngroups && row < a.nrows) {
            const cx<T>* src = reinterpret_cast<const cx<T>*>(in + row * a.real_rs) + tp;
            static_for<NLOAD>([&](auto ic) {
                constexpr int n1 = decltype(ic)::value;
                dst[n1] = (!PRUNE || tp + R2 * n1 < a.nc) ? src[R2 * n1] : cx<T>{0, 0};
            });
        } else {
            static_for<NLOAD>([&](auto ic) { dst[decltype(ic)::value] = cx<T>{0, 0}; });
        }
    };
    constexpr bool PF = PRUNE;           // a full-length row (periodic axis) leaves no registers for the prefetch
    cx<T> vn[PF ? NLOAD : 1];
    if constexpr (PF) fetch(blockIdx.x, vn);
    {
        const cx<T>* twg = static_cast<const cx<T>*>(a.tw);
        // tw[k1 * R2 + n2] = w_M^(n2 k1): the R2 threads of a row read consecutive entries (no bank conflicts)
        for (int e = threadIdx.x; e < M; e += 256) {
            tw[e] = twg[((e / R2) * (e % R2)) * (kTwiddleN / M)];
            tws[e] = twg[e * (kTwiddleN / (2 * M))];
        }
    }
    __syncthreads();
    for (int64_t grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
        const int64_t row = grp * C::ROWS + rl;
        const bool live = row < a.nrows;
        cx<T> v[R1];
        if constexpr (PF) {
            static_for<NLOAD>([&](auto ic) { v[decltype(ic)::value] = vn[decltype(ic)::value]; });
            fetch(grp + gridDim.x, vn);
        } else {
            fetch(grp, v);
        }
        Dif<T, -1, R1, 0, PRUNE>::run(v);
        static_for<R1>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            constexpr int k1 = brev<R1>(p);
            cx<T> val = v[p];
            if constexpr (k1 != 0) val = cmul(val, tw[k1 * R2 + tp]);
            rb[k1 * (R2 + 1) + tp] = val;
        });
        __syncthreads();
        cx<T> u[NT3][R2];
#pragma unroll
        for (int it = 0; it < NT3; ++it) {
            const int k1 = tp + it * TPP;
            static_for<R2>([&](auto nc) { u[it][decltype(nc)::value] = rb[k1 * (R2 + 1) + decltype(nc)::value]; });
            Dif<T, -1, R2>::run(u[it]);
        }
        __syncthreads();     // exchange layout fully read; reuse the row buffer in natural order
#pragma unroll
        for (int it = 0; it < NT3; ++it) {
            const int k1 = tp + it * TPP;
            static_for<R2>([&](auto pc) {
                constexpr int p = decltype(pc)::value;
                rb[k1 + R1 * brev<R2>(p)] = u[it][p];
            });
        }
        __syncthreads();
        if (live) {
            cx<T>* dst = out + spec_row(a, row);
            for (int k = tp; k <= M / 2; k += TPP) {
                const cx<T> Zk = rb[k], Zn = rb[(M - k) & (M - 1)];
                const T ex = (T)0.5 * (Zk.x + Zn.x), ey = (T)0.5 * (Zk.y - Zn.y);
                const T ox = (T)0.5 * (Zk.y + Zn.y), oy = (T)-0.5 * (Zk.x - Zn.x);
                const cx<T> w = tws[k];
                // X[k] = Xe + w Xo;  X[M-k] = conj(Xe) - conj(w Xo)   (w_2M^(M-k) = -conj(w_2M^k), Xo(M-k) = conj Xo(k))
                const T px = ox * w.x - oy * w.y, py = ox * w.y + oy * w.x;
                dst[spec_off(a, k)] = {ex + px, ey + py};
                dst[spec_off(a, M - k)] = {ex - px, py - ey};
            }
        }
        __syncthreads();     // row buffer fully read before the next group's exchange is written
    }
}

template <typename T, int M, bool PRUNE>
__global__ void __launch_bounds__(256, M >= 512 ? 1 : 2) k2_xinv(const cx<T>* __restrict__ in, T* __restrict__ out, X2Args a)
{
    using C = XCfg<M>;
    constexpr int R1 = C::R1, R2 = C::R2, TPP = C::TPP, NT3 = R1 / TPP, TWG = R1 < 8 ? R1 : 8;
    cx<T>* tw = reinterpret_cast<cx<T>*>(fe2_smem);
    cx<T>* tws = tw + M;
    cx<T>* buf = tws + M;
    const int tp = threadIdx.x % TPP, rl = threadIdx.x / TPP;
    const int64_t row = (int64_t)blockIdx.x * C::ROWS + rl;
    const bool live = row < a.nrows;
    cx<T>* rb = buf + rl * C::RPITCH;

    {
        const cx<T>* twg = static_cast<const cx<T>*>(a.tw);
        // tw[k1 * R2 + n2] = w_M^(n2 k1): the R2 threads of a row read consecutive entries (no bank conflicts)
        for (int e = threadIdx.x; e < M; e += 256) {
            tw[e] = twg[((e / R2) * (e % R2)) * (kTwiddleN / M)];
            tws[e] = twg[e * (kTwiddleN / (2 * M))];
        }
    }
    __syncthreads();
    cx<T> v[R1];
    const cx<T>* src = in + spec_row(a, live ? row : 0);
    static_for<R1>([&](auto jc) {
        constexpr int j1 = decltype(jc)::value;
        const int k = tp + R2 * j1;
        const cx<T> Xk = src[spec_off(a, k)], Xn = src[spec_off(a, M - k)];
        const T ex = (T)0.5 * (Xk.x + Xn.x), ey = (T)0.5 * (Xk.y - Xn.y);
        const T dx = (T)0.5 * (Xk.x - Xn.x), dy = (T)0.5 * (Xk.y + Xn.y);
        const cx<T> w = tws[k];
        const T ox = dx * w.x + dy * w.y, oy = dy * w.x - dx * w.y;   // D * conj(w)
        v[j1] = {ex - oy, ey + ox};
    });
    Dif<T, +1, R1>::run(v);
    // twiddles are fetched in groups of TWG ahead of the stores they feed: a load from the table cannot be moved
    // above a store to the row buffer by the compiler (both are shared memory).  (The forward kernel is bound by
    // shared-memory throughput, not latency, and is faster with the loads left where they are used.)
    static_for<R1 / TWG>([&](auto gc) {
        constexpr int g = decltype(gc)::value;
        cx<T> w[TWG];
        static_for<TWG>([&](auto qc) {
            constexpr int o1 = brev<R1>(g * TWG + decltype(qc)::value);
            if constexpr (o1 != 0) w[decltype(qc)::value] = tw[o1 * R2 + tp];
        });
        static_for<TWG>([&](auto qc) {
            constexpr int p = g * TWG + decltype(qc)::value;
            constexpr int o1 = brev<R1>(p);
            cx<T> val = v[p];
            if constexpr (o1 != 0) val = cmulc(val, w[decltype(qc)::value]);
            rb[o1 * (R2 + 1) + tp] = val;
        });
    });
    __syncthreads();
#pragma unroll
    for (int it = 0; it < NT3; ++it) {
        const int o1 = tp + it * TPP;
        cx<T> u[R2];
        static_for<R2>([&](auto nc) { u[decltype(nc)::value] = rb[o1 * (R2 + 1) + decltype(nc)::value]; });
        Dif<T, +1, R2>::run(u);
        if (live) {
            cx<T>* dst = reinterpret_cast<cx<T>*>(out + row * a.real_rs) + o1;
            static_for<R2>([&](auto pc) {
                constexpr int p = decltype(pc)::value;
                constexpr int o2 = brev<R2>(p);
                if constexpr (!PRUNE || o2 < R2 / 2) {
                    if (!PRUNE || o1 + R1 * o2 < a.nc) dst[R1 * o2] = u[p];
                }
            });
        }
    }
}

template <typename T, int M, bool PRUNE, bool FWD>
static cudaError_t launch_one(const void* in, void* out, const X2Args& a, cudaStream_t st)
{
    using C = XCfg<M>;
    constexpr size_t smem = (size_t)(2 * M + C::ROWS * C::RPITCH) * sizeof(cx<T>);
    const dim3 grid((unsigned)((a.nrows + C::ROWS - 1) / C::ROWS));
    if constexpr (FWD) {
        // persistent: as many blocks as fit on the device (rows are visited with a grid stride)
        static PerDevice<int> cache;
        int& nblocks = cache.here();
        if (!nblocks) {
            cudaError_t e = cudaFuncSetAttribute(k2_xfwd<T, M, PRUNE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
            int dev = 0, sms = 0, per = 0;
            if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
            if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
            if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, k2_xfwd<T, M, PRUNE>, 256, smem)) != cudaSuccess) return e;
            nblocks = sms * (per > 0 ? per : 1);
        }
        const dim3 pgrid(grid.x < (unsigned)nblocks ? grid.x : (unsigned)nblocks);
        k2_xfwd<T, M, PRUNE><<<pgrid, 256, smem, st>>>(static_cast<const T*>(in), static_cast<cx<T>*>(out), a);
    } else {
        static PerDevice<int> cache;
        int& configured = cache.here();
        if (!configured) {
            cudaError_t e = cudaFuncSetAttribute(k2_xinv<T, M, PRUNE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
            configured = 1;
        }
        k2_xinv<T, M, PRUNE><<<grid, 256, smem, st>>>(static_cast<const cx<T>*>(in), static_cast<T*>(out), a);
    }
    return cudaGetLastError();
}

template <typename T, bool FWD>
static cudaError_t launch_x(int M, bool prune, const void* in, void* out, const X2Args& a, cudaStream_t st)
{
    switch (M) {
        case 64: return prune ? launch_one<T, 64, true, FWD>(in, out, a, st) : launch_one<T, 64, false, FWD>(in, out, a, st);
        case 128: return prune ? launch_one<T, 128, true, FWD>(in, out, a, st) : launch_one<T, 128, false, FWD>(in, out, a, st);
        case 256: return prune ? launch_one<T, 256, true, FWD>(in, out, a, st) : launch_one<T, 256, false, FWD>(in, out, a, st);
        case 512: return prune ? launch_one<T, 512, true, FWD>(in, out, a, st) : launch_one<T, 512, false, FWD>(in, out, a, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace v2

bool x2_supported(int Mc) { return Mc == 64 || Mc == 128 || Mc == 256 || Mc == 512; }

// nrows real rows of n_real valid reals (n_real == 2 Mc, or Mc when zero-padded), real_rs apart; spectrum strides
// spec[4] = { ny (rows per plane), s_plane, s_row, s_g } as in X2Args, lanes = kx per group (power of two)
template <typename T>
cudaError_t launch_xfwd2(const FftCtx& c, const T* in, void* out, int n_real, int64_t nrows, int64_t real_rs,
                         const int64_t spec[4], int lanes, cudaStream_t st)
{
    const int M = c.plan[0].M;
    const bool prune = n_real <= M;          // zero-padded axis: at most half of the 2 M reals are data
    if ((!prune && n_real != 2 * M) || (n_real & 1)) return cudaErrorInvalidValue;
    int lg = 0;
    while ((1 << lg) < lanes) ++lg;
    v2::X2Args a{c.tw, nrows, real_rs, (int)spec[0], lg, spec[1], spec[2], spec[3], n_real / 2};
    return v2::launch_x<T, true>(M, prune, in, out, a, st);
}

template <typename T>
cudaError_t launch_xinv2(const FftCtx& c, const void* in, T* out, int n_real, int64_t nrows, int64_t real_rs,
                         const int64_t spec[4], int lanes, cudaStream_t st)
{
    const int M = c.plan[0].M;
    const bool prune = n_real <= M;          // zero-padded axis: at most half of the 2 M reals are data
    if ((!prune && n_real != 2 * M) || (n_real & 1)) return cudaErrorInvalidValue;
    int lg = 0;
    while ((1 << lg) < lanes) ++lg;
    v2::X2Args a{c.tw, nrows, real_rs, (int)spec[0], lg, spec[1], spec[2], spec[3], n_real / 2};
    return v2::launch_x<T, false>(M, prune, in, out, a, st);
}

template cudaError_t launch_xfwd2<double>(const FftCtx&, const double*, void*, int, int64_t, int64_t, const int64_t*, int, cudaStream_t);
template cudaError_t launch_xfwd2<float>(const FftCtx&, const float*, void*, int, int64_t, int64_t, const int64_t*, int, cudaStream_t);
template cudaError_t launch_xinv2<double>(const FftCtx&, const void*, double*, int, int64_t, int64_t, const int64_t*, int, cudaStream_t);
template cudaError_t launch_xinv2<float>(const FftCtx&, const void*, float*, int, int64_t, int64_t, const int64_t*, int, cudaStream_t);

}  // namespace fe
