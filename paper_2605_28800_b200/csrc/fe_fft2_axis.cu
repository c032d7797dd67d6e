// fe_fft2_axis.cu -- size-specialised strided pass along y:
// forward reads n_keep rows (the rest of the padded axis is zero) and writes M rows, inverse reads M rows and
// writes n_keep rows.  A tile is M rows x 128 bytes of consecutive kx; the transform runs in registers with
// one shared-memory exchange (fe_fft2.cuh).
#include "fe_fft2.cuh"

namespace fe {
namespace v2 {

// A tile is M rows of LANES consecutive complex elements.  Its first element sits at
// blockIdx.x * s0 + blockIdx.y * s1 + blockIdx.z * sb, its rows are sa apart (all in complex elements), so the
// same kernels serve the row-major spectra and the tiled layouts of fe_api.cu.
struct Axis2Args {
    const void* tw;
    int n_keep;       // rows that carry data on the pruned side (<= M/2 on a zero-padded axis)
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
        v[n1] = (!PIN || row < a.n_keep) ? ib[(int64_t)row * a.in_sa] : cx<T>{0, 0};
    });
    load_twiddles<T, M>(tw, static_cast<const cx<T>*>(a.tw), threadIdx.x, LANES * TPP);
    __syncthreads();
    Dif<T, DIR, R1, 0, PIN>::run(v);
    // twiddles are fetched in groups ahead of the stores they feed (a shared-memory load cannot be moved above a
    // shared-memory store by the compiler)
    constexpr int TWG = R1 < 8 ? R1 : 8;
    static_for<R1 / TWG>([&](auto gc) {
        constexpr int g = decltype(gc)::value;
        cx<T> w[TWG];
        static_for<TWG>([&](auto qc) {
            constexpr int k1 = brev<R1>(g * TWG + decltype(qc)::value);
            if constexpr (k1 != 0) w[decltype(qc)::value] = tw[tp * k1];
        });
        static_for<TWG>([&](auto qc) {
            constexpr int p = g * TWG + decltype(qc)::value;
            constexpr int k1 = brev<R1>(p);
            cx<T> val = v[p];
            if constexpr (k1 != 0) val = cmuld<T, DIR>(val, w[decltype(qc)::value]);
            buf[(k1 * R2 + tp) * LANES + lane] = val;
        });
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
                if (!POUT || row < a.n_keep) ob[(int64_t)row * a.out_sa] = u[p];
            }
        });
    }
}

// Three-level factorisation of the long axes (M = 256, 512): M = RA * RB * RC,
//   n = n3 + RC n2 + RC RB n1,   k = k1 + RA k2 + RA RB k3,
//   A: RA-point over n1, twiddle w_M^((n3 + RC n2) k1);  B: RB-point over n2 (in place), twiddle w_M^(RA n3 k2);
//   C: RC-point over n3.
// A thread holds at most 8 points, so a 256-thread block needs ~80 registers per thread.
template <int M> struct Fact3;
template <> struct Fact3<256> { static constexpr int RA = 8, RB = 8, RC = 4; };
template <> struct Fact3<512> { static constexpr int RA = 8, RB = 8, RC = 8; };

// ------------------------------------------------------------------------------------------------
// Bulk-copy variant for contiguous tiles (tiled layouts of fe_api.cu, M = 256 or 512): persistent blocks, a ring
// of three M x 128-byte buffers per block.  A tile arrives with one cp.async.bulk (mbarrier completion), is
// transformed IN PLACE by the three-level scheme above (every task writes exactly the slots it read), and leaves
// with one cp.async.bulk store, so loads of tile i+2, the transform of tile i and the store of tile i-1 overlap
// and no data passes through registers on its way to or from HBM.
//   forward: input row y at slot y; output frequency k = k1 + RA k2 + RA RB k3 at slot (k1 RB + k2) RC + k3
//            ("slot order": the digit-reversed ky order in which S2 is stored when this kernel is used),
//   inverse: input in slot order, levels run C', B', A'; output row y at slot y.
// ------------------------------------------------------------------------------------------------
struct Axis4Args {
    const void* tw;
    int n0, n1, ntiles;                   // tile t -> (t % n0, (t / n0) % n1, t / (n0 n1))
    int n_keep;                           // data rows on the pruned side (<= M/2)
    int64_t in_s0, in_s1, in_sb, out_s0, out_s1, out_sb;
};

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(void* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(void* bar, unsigned parity)
{
    const unsigned addr = smem_u32(bar);
    unsigned done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(addr), "r"(parity)
            : "memory");
    } while (!done);
}
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gsrc, unsigned bytes, void* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void bulk_store(void* gdst, const void* smem_src, unsigned bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;\n" ::"l"(gdst), "r"(smem_u32(smem_src)),
                 "r"(bytes)
                 : "memory");
    asm volatile("cp.async.bulk.commit_group;\n" ::: "memory");
}
template <int N> __device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;\n" ::"n"(N) : "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }

template <typename T, int M, int DIR, bool PRUNE, int THREADS>
__global__ void __launch_bounds__(THREADS, 1)
k4_axis(const cx<T>* __restrict__ in, cx<T>* __restrict__ out, Axis4Args a)
{
    constexpr int RA = Fact3<M>::RA, RB = Fact3<M>::RB, RC = Fact3<M>::RC;
    constexpr int LANES = 128 / (int)sizeof(cx<T>);
    constexpr int TPP = THREADS / LANES;
    constexpr int NTA = RB * RC, NTB = RA * RC, NTC = RA * RB;
    static_assert(NTA % TPP == 0 && NTB % TPP == 0 && NTC % TPP == 0, "tasks must divide evenly");
    constexpr int NB = 3;
    constexpr int TILE = M * LANES;
    constexpr bool PIN = PRUNE && DIR < 0, POUT = PRUNE && DIR > 0;
    const unsigned in_bytes = (unsigned)((PIN ? a.n_keep : M) * LANES * sizeof(cx<T>));
    const unsigned out_bytes = (unsigned)((POUT ? a.n_keep : M) * LANES * sizeof(cx<T>));
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(fe2_smem);     // [NB], 64 bytes reserved
    cx<T>* tw = reinterpret_cast<cx<T>*>(fe2_smem + 64);
    cx<T>* bufs = tw + M;
    const int lane = threadIdx.x % LANES, tp = threadIdx.x / LANES;

    auto in_ptr = [&](int t) {
        const int i0 = t % a.n0, r = t / a.n0, i1 = r % a.n1, ib = r / a.n1;
        return in + (int64_t)ib * a.in_sb + (int64_t)i1 * a.in_s1 + (int64_t)i0 * a.in_s0;
    };
    auto out_ptr = [&](int t) {
        const int i0 = t % a.n0, r = t / a.n0, i1 = r % a.n1, ib = r / a.n1;
        return out + (int64_t)ib * a.out_sb + (int64_t)i1 * a.out_s1 + (int64_t)i0 * a.out_s0;
    };
    if (threadIdx.x == 0) {
        for (int b = 0; b < NB; ++b) mbar_init(&bars[b], 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    load_twiddles<T, M>(tw, static_cast<const cx<T>*>(a.tw), threadIdx.x, THREADS);
    __syncthreads();
    const int t0 = blockIdx.x, dt = gridDim.x;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int pre = 0; pre < 2; ++pre) {
            const int t = t0 + pre * dt;
            if (t < a.ntiles) {
                mbar_expect_tx(&bars[pre], in_bytes);
                bulk_load(bufs + pre * TILE, in_ptr(t), in_bytes, &bars[pre]);
            }
        }
    }
    // Inter-level twiddles of this thread's tasks.  They do not depend on the tile, and a load from the table
    // cannot be moved above a store to the tile by the compiler (both live in shared memory), so loading them
    // where they are used puts one shared-memory latency between every two stores.  With 256 threads they stay in
    // registers for the whole kernel; the 512-thread variant reloads them at the top of every tile.
    static_assert(TPP % RB == 0 && TPP % RC == 0, "digits of a task must not depend on the task round");
    constexpr bool HOIST = THREADS <= 256;
    constexpr int NWA = DIR < 0 ? NTA / TPP : NTB / TPP;
    cx<T> w1[NWA][8];                    // forward: level A, tw[j k1];       inverse: level B', tw[(n3 + RC n2) k1]
    cx<T> w2[8];                         // forward: level B, tw[RA n3 k2];   inverse: level C', tw[RA n3 k2]
    auto load_tw = [&]() {
        if (DIR < 0) {
#pragma unroll
            for (int it = 0; it < NTA / TPP; ++it) {
                const int j = tp + it * TPP;
                static_for<RA - 1>([&](auto kc) { w1[it][decltype(kc)::value + 1] = tw[j * (decltype(kc)::value + 1)]; });
            }
            const int n3 = tp % RC;
            static_for<RB - 1>([&](auto kc) { w2[decltype(kc)::value + 1] = tw[RA * n3 * (decltype(kc)::value + 1)]; });
        } else {
            const int k2 = tp % RB;
            static_for<RC - 1>([&](auto nc) { w2[decltype(nc)::value + 1] = tw[RA * (decltype(nc)::value + 1) * k2]; });
#pragma unroll
            for (int it = 0; it < NTB / TPP; ++it) {
                const int tb = tp + it * TPP, n3 = tb % RC, k1 = tb / RC;
                static_for<RB>([&](auto nc) { w1[it][decltype(nc)::value] = tw[(n3 + RC * decltype(nc)::value) * k1]; });
            }
        }
    };
    if (HOIST) load_tw();
    // The buffer of tile i-1 is reused for tile i+2: its store must have finished reading shared memory.  Issued
    // by thread 0 after the first level of tile i (the store of tile i-1 is the newest bulk group then), which gives
    // the load two thirds of a tile more lead than issuing it behind the store of tile i.
    auto prefetch_next = [&](int t, int i) {
        const int tn = t + 2 * dt;
        if (tn < a.ntiles) {
            bulk_wait_read<0>();
            const int bn = (i + 2) % NB;
            mbar_expect_tx(&bars[bn], in_bytes);
            bulk_load(bufs + bn * TILE, in_ptr(tn), in_bytes, &bars[bn]);
        }
    };
    int i = 0;
    for (int t = t0; t < a.ntiles; t += dt, ++i) {
        const int b = i % NB;
        cx<T>* buf = bufs + b * TILE + lane;
        if (!HOIST) load_tw();
        mbar_wait(&bars[b], (unsigned)((i / NB) & 1));
        if (PIN && a.n_keep < M / 2) {
            // the zero padding below M/2 is not part of the tile in memory: clear the rows the previous tile left there
            for (int e = a.n_keep * LANES + threadIdx.x; e < (M / 2) * LANES; e += THREADS) bufs[b * TILE + e] = cx<T>{0, 0};
            __syncthreads();
        }
        if (DIR < 0) {
            // ---- A: task j = n3 + RC n2, slots j + RB RC n1
#pragma unroll
            for (int it = 0; it < NTA / TPP; ++it) {
                const int j = tp + it * TPP;
                cx<T> u[RA];
                cx<T>* col = buf + j * LANES;
                static_for<(PIN ? RA / 2 : RA)>([&](auto ic) { u[decltype(ic)::value] = col[decltype(ic)::value * RB * RC * LANES]; });
                Dif<T, DIR, RA, 0, PIN>::run(u);
                static_for<RA>([&](auto pc) {
                    constexpr int p = decltype(pc)::value;
                    constexpr int k1 = brev<RA>(p);
                    cx<T> val = u[p];
                    if constexpr (k1 != 0) val = cmul(val, w1[it][k1]);
                    col[k1 * RB * RC * LANES] = val;
                });
            }
            __syncthreads();
            if (threadIdx.x == 0) prefetch_next(t, i);
            // ---- B: task (k1, n3), slots k1 RB RC + n3 + RC n2
#pragma unroll
            for (int it = 0; it < NTB / TPP; ++it) {
                const int tb = tp + it * TPP, n3 = tb % RC, k1 = tb / RC;
                cx<T> u[RB];
                cx<T>* col = buf + (k1 * RB * RC + n3) * LANES;
                static_for<RB>([&](auto nc) { u[decltype(nc)::value] = col[decltype(nc)::value * RC * LANES]; });
                Dif<T, DIR, RB>::run(u);
                static_for<RB>([&](auto pc) {
                    constexpr int p = decltype(pc)::value;
                    constexpr int k2 = brev<RB>(p);
                    cx<T> val = u[p];
                    if constexpr (k2 != 0) val = cmul(val, w2[k2]);
                    col[k2 * RC * LANES] = val;
                });
            }
            __syncthreads();
            // ---- C: task tc = k1 RB + k2, slots tc RC + n3
#pragma unroll
            for (int it = 0; it < NTC / TPP; ++it) {
                const int tc = tp + it * TPP;
                cx<T> u[RC];
                cx<T>* col = buf + tc * RC * LANES;
                static_for<RC>([&](auto nc) { u[decltype(nc)::value] = col[decltype(nc)::value * LANES]; });
                Dif<T, DIR, RC>::run(u);
                static_for<RC>([&](auto pc) { col[brev<RC>(decltype(pc)::value) * LANES] = u[decltype(pc)::value]; });
            }
        } else {
            // ---- C': task tc = k1 RB + k2 (k2 = tc % RB), slots tc RC + k3 -> n3
#pragma unroll
            for (int it = 0; it < NTC / TPP; ++it) {
                const int tc = tp + it * TPP, k2 = tc % RB;
                cx<T> u[RC];
                cx<T>* col = buf + tc * RC * LANES;
                static_for<RC>([&](auto nc) { u[decltype(nc)::value] = col[decltype(nc)::value * LANES]; });
                Dif<T, DIR, RC>::run(u);
                static_for<RC>([&](auto pc) {
                    constexpr int p = decltype(pc)::value;
                    constexpr int n3 = brev<RC>(p);
                    cx<T> val = u[p];
                    if constexpr (n3 != 0) val = cmulc(val, w2[n3]);
                    col[n3 * LANES] = val;
                });
            }
            __syncthreads();
            if (threadIdx.x == 0) prefetch_next(t, i);
            // ---- B': task (k1, n3), slots k1 RB RC + n3 + RC k2 -> n2
#pragma unroll
            for (int it = 0; it < NTB / TPP; ++it) {
                const int tb = tp + it * TPP, n3 = tb % RC, k1 = tb / RC;
                cx<T> u[RB];
                cx<T>* col = buf + (k1 * RB * RC + n3) * LANES;
                static_for<RB>([&](auto nc) { u[decltype(nc)::value] = col[decltype(nc)::value * RC * LANES]; });
                Dif<T, DIR, RB>::run(u);
                static_for<RB>([&](auto pc) {
                    constexpr int p = decltype(pc)::value;
                    constexpr int n2 = brev<RB>(p);
                    col[n2 * RC * LANES] = cmulc(u[p], w1[it][n2]);
                });
            }
            __syncthreads();
            // ---- A': task j = n3 + RC n2, slots j + RB RC k1 -> n1 (first half kept when pruned)
#pragma unroll
            for (int it = 0; it < NTA / TPP; ++it) {
                const int j = tp + it * TPP;
                cx<T> u[RA];
                cx<T>* col = buf + j * LANES;
                static_for<RA>([&](auto kc) { u[decltype(kc)::value] = col[decltype(kc)::value * RB * RC * LANES]; });
                Dif<T, DIR, RA>::run(u);
                static_for<RA>([&](auto pc) {
                    constexpr int p = decltype(pc)::value;
                    constexpr int n1 = brev<RA>(p);
                    if constexpr (!POUT || n1 < RA / 2) col[n1 * RB * RC * LANES] = u[p];
                });
            }
        }
        fence_async_smem();                 // generic-proxy writes of this thread -> visible to the bulk store
        __syncthreads();
        if (threadIdx.x == 0) {
            bulk_store(out_ptr(t), bufs + b * TILE, out_bytes);
        }
    }
    if (threadIdx.x == 0) bulk_wait_read<0>();
}

template <typename T, int M, int DIR, bool PRUNE, int THREADS>
static cudaError_t launch_one4(const void* in, void* out, Axis4Args a, cudaStream_t st)
{
    constexpr int LANES = 128 / (int)sizeof(cx<T>);
    constexpr size_t smem = 64 + (size_t)(M + 3 * M * LANES) * sizeof(cx<T>);
    static PerDevice<int> cache;
    int& nblocks = cache.here();
    if (!nblocks) {
        cudaError_t e = cudaFuncSetAttribute(k4_axis<T, M, DIR, PRUNE, THREADS>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        int dev = 0, sms = 0, per = 0;
        if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, k4_axis<T, M, DIR, PRUNE, THREADS>, THREADS, smem)) !=
            cudaSuccess)
            return e;
        nblocks = sms * (per > 0 ? per : 1);
    }
    const int grid = a.ntiles < nblocks ? a.ntiles : nblocks;
    k4_axis<T, M, DIR, PRUNE, THREADS><<<grid, THREADS, smem, st>>>(static_cast<const cx<T>*>(in), static_cast<cx<T>*>(out), a);
    return cudaGetLastError();
}

template <typename T, int M, int THREADS>
static cudaError_t launch_m4(int dir, bool prune, const void* in, void* out, const Axis4Args& a, cudaStream_t st)
{
    if (dir < 0) return prune ? launch_one4<T, M, -1, true, THREADS>(in, out, a, st)
                              : launch_one4<T, M, -1, false, THREADS>(in, out, a, st);
    return prune ? launch_one4<T, M, +1, true, THREADS>(in, out, a, st) : launch_one4<T, M, +1, false, THREADS>(in, out, a, st);
}

template <typename T, int M, int DIR, bool PRUNE>
static cudaError_t launch_one(const void* in, void* out, const Axis2Args& a, dim3 grid, cudaStream_t st)
{
    constexpr int LANES = 128 / (int)sizeof(cx<T>);
    constexpr int threads = LANES * Fact<M>::R2;
    constexpr size_t smem = (size_t)(M + M * LANES) * sizeof(cx<T>);
    static PerDevice<int> cache;
    int& configured = cache.here();
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(k2_axis<T, M, DIR, PRUNE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)smem);
        if (e != cudaSuccess) return e;
        configured = 1;
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
    v2::Axis2Args a{c.tw, n_keep, in_sa, in_s0, in_s1, in_sb, out_sa, out_s0, out_s1, out_sb};
    dim3 grid(n0, n1, batch);
    const bool prune = 2 * n_keep <= M;          // zero-padded axis
    if (!prune && n_keep != M) return cudaErrorInvalidValue;
    switch (M) {
        case 64: return v2::launch_m<T, 64>(dir, prune, in, out, a, grid, st);
        case 128: return v2::launch_m<T, 128>(dir, prune, in, out, a, grid, st);
        case 256: return v2::launch_m<T, 256>(dir, prune, in, out, a, grid, st);
        case 512: return v2::launch_m<T, 512>(dir, prune, in, out, a, grid, st);
        default: return cudaErrorInvalidValue;
    }
}

bool axis4_supported(int M) { return M == 256 || M == 512; }

// slot of frequency k in the output of the bulk-copy pass (and of its input in the inverse direction)
int axis4_slot(int M, int k)
{
    int RA, RB, RC;
    if (M == 512) { RA = v2::Fact3<512>::RA; RB = v2::Fact3<512>::RB; RC = v2::Fact3<512>::RC; }
    else { RA = v2::Fact3<256>::RA; RB = v2::Fact3<256>::RB; RC = v2::Fact3<256>::RC; }
    const int k1 = k % RA, k2 = (k / RA) % RB, k3 = k / (RA * RB);
    return (k1 * RB + k2) * RC + k3;
}
void axis4_radices(int M, int r[3])
{
    if (M == 512) { r[0] = v2::Fact3<512>::RA; r[1] = v2::Fact3<512>::RB; r[2] = v2::Fact3<512>::RC; }
    else { r[0] = v2::Fact3<256>::RA; r[1] = v2::Fact3<256>::RB; r[2] = v2::Fact3<256>::RC; }
}

// Bulk-copy pass over contiguous tiles: tile (i0, i1, ib) of the input starts at i0 in_s0 + i1 in_s1 + ib in_sb and
// holds n_keep (forward) or M (inverse) rows of 128 bytes back to back; the output tile likewise.  The spectrum
// side is in slot order (axis4_slot).
template <typename T>
cudaError_t launch_axis4(const FftCtx& c, int axis, int dir, const void* in, void* out, int n_keep, int n0, int n1,
                         int batch, int64_t in_s0, int64_t in_s1, int64_t in_sb, int64_t out_s0, int64_t out_s1,
                         int64_t out_sb, cudaStream_t st)
{
    const int M = c.plan[axis].M;
    const bool prune = 2 * n_keep <= M;          // zero-padded axis
    if (!prune && n_keep != M) return cudaErrorInvalidValue;
    v2::Axis4Args a{c.tw, n0, n1, n0 * n1 * batch, n_keep, in_s0, in_s1, in_sb, out_s0, out_s1, out_sb};
    if (M == 256) return v2::launch_m4<T, 256, 256>(dir, prune, in, out, a, st);
    if (M == 512) return v2::launch_m4<T, 512, 256>(dir, prune, in, out, a, st);
    return cudaErrorInvalidValue;
}

template cudaError_t launch_axis4<double>(const FftCtx&, int, int, const void*, void*, int, int, int, int, int64_t,
                                          int64_t, int64_t, int64_t, int64_t, int64_t, cudaStream_t);
template cudaError_t launch_axis4<float>(const FftCtx&, int, int, const void*, void*, int, int, int, int, int64_t,
                                         int64_t, int64_t, int64_t, int64_t, int64_t, cudaStream_t);

template cudaError_t launch_axis2<double>(const FftCtx&, int, int, const void*, void*, int, int, int, int, int64_t,
                                          int64_t, int64_t, int64_t, int64_t, int64_t, int64_t, int64_t, cudaStream_t);
template cudaError_t launch_axis2<float>(const FftCtx&, int, int, const void*, void*, int, int, int, int, int64_t,
                                         int64_t, int64_t, int64_t, int64_t, int64_t, int64_t, int64_t, cudaStream_t);

}  // namespace fe
