// fe_fft2_xy.cu -- x and y passes fused through an L2-resident ring of S1 planes (the
// "504 B" row of 8(d); "dominant computational cost").
//
// The two-kernel path writes the half spectrum S1 of every z plane to HBM after the x pass and reads it back in the
// y pass (2 x 3 s p_x bytes per cell and direction).  Here ONE cooperative persistent kernel runs both passes:
//   X group (256 threads of every block): x pass of ROWS rows at a time, output into slot (plane mod RING) of a small
//            ring of S1 planes (a few MB: stays in the 126 MB L2, its lines are overwritten before they are evicted);
//   Y group (the other 256 threads): bulk-copy three-level y pass of the tiles of a plane once all its rows are there.
// Planes are produced and consumed in the same order; per-plane counters in global memory order the two groups:
//   xdone[p]  rows groups of plane p written           (Y tile of plane p waits for xdone[p] == groups per plane)
//   ydone[p]  tiles of plane p read                     (X rows of plane p wait for ydone[p - RING] == tiles per plane)
// Every wait points to work that comes EARLIER in the same order and all blocks are co-resident (cooperative launch),
// so the kernel cannot deadlock; a spin that exceeds ~1 s of clock ticks raises an error flag and gives up.
// The inverse kernel mirrors this: Y group (inverse y pass) produces ring planes, X group (inverse x pass) consumes.
#include "fe_fft2.cuh"

namespace fe {
namespace v2 {

struct XYArgs {
    const void* tw;            // 2048-entry forward twiddle table
    int nplanes;               // batch * 3 * nz
    int nz, ny, G, ring;       // rows per plane, kx groups per plane, ring slots
    int nc;                    // valid complex pairs per real row (n_x / 2)
    int lg;                    // log2(kx per group)
    int xgroups;               // row groups per plane (ny / ROWS)
    int64_t real_rs;           // real row stride (n_x)
    int64_t ring_plane;        // complex elements of one ring plane: G * ny * L
    int64_t s2_sz, s2_sg, s2_sb;   // S2 tile (bc, z, g) starts at bc * s2_sb + z * s2_sz + g * s2_sg
    int* xdone;                // [nplanes], zeroed before the launch
    int* ydone;                // [nplanes]
    int* err;                  // set to 1 when a wait timed out
};

__device__ __forceinline__ unsigned xy_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void xy_bar(int id) { asm volatile("bar.sync %0, 256;\n" ::"r"(id) : "memory"); }
__device__ __forceinline__ int xy_ld_acquire(const int* p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void xy_red_release(int* p)
{
    asm volatile("red.release.gpu.global.add.s32 [%0], 1;\n" ::"l"(p) : "memory");
}
__device__ __forceinline__ void xy_fence_proxy() { asm volatile("fence.proxy.async.global;\n" ::: "memory"); }
// spin until *p >= target; false (and *err = 1) after ~2^31 clock ticks
__device__ __forceinline__ bool xy_wait(const int* p, int target, int* err)
{
    if (xy_ld_acquire(p) >= target) return true;
    const long long t0 = clock64();
    while (xy_ld_acquire(p) < target) {
        __nanosleep(100);
        if (*reinterpret_cast<volatile int*>(err)) return false;       // another wait gave up: do not wait again
        if (clock64() - t0 > (1ll << 31)) {
            *err = 1;
            return false;
        }
    }
    return true;
}
__device__ __forceinline__ void xy_mbar_init(void* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(xy_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void xy_mbar_expect_tx(void* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(xy_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void xy_mbar_wait(void* bar, unsigned parity)
{
    const unsigned addr = xy_smem_u32(bar);
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
__device__ __forceinline__ void xy_bulk_load(void* smem_dst, const void* gsrc, unsigned bytes, void* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(
                     xy_smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(xy_smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void xy_bulk_store(void* gdst, const void* smem_src, unsigned bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;\n" ::"l"(gdst), "r"(xy_smem_u32(smem_src)),
                 "r"(bytes)
                 : "memory");
    asm volatile("cp.async.bulk.commit_group;\n" ::: "memory");
}
template <int N> __device__ __forceinline__ void xy_bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;\n" ::"n"(N) : "memory"); }
template <int N> __device__ __forceinline__ void xy_bulk_wait_all() { asm volatile("cp.async.bulk.wait_group %0;\n" ::"n"(N) : "memory"); }
__device__ __forceinline__ void xy_fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }

template <int M> struct XYFact3;
template <> struct XYFact3<256> { static constexpr int RA = 8, RB = 8, RC = 4; };
template <> struct XYFact3<512> { static constexpr int RA = 8, RB = 8, RC = 8; };

// shared-memory plan of one block
template <typename T, int MX, int MY> struct XYCfg {
    static constexpr int R1 = Fact<MX>::R1, R2 = Fact<MX>::R2;
    static constexpr int ROWS = 256 / R2;                                   // rows per X task
    static constexpr int XPITCH = R1 * (R2 + 1);
    static constexpr int RPITCH = XPITCH > MX + 1 ? XPITCH : MX + 1;
    static constexpr int LANES = 128 / (int)sizeof(cx<T>);
    static constexpr int TILE = MY * LANES;                                 // complex elements of a y tile
    static constexpr size_t x_bytes = (size_t)(2 * MX + ROWS * RPITCH) * sizeof(cx<T>);
    static constexpr size_t ytw_bytes = (size_t)MY * sizeof(cx<T>);
    static constexpr size_t tile_bytes = (size_t)TILE * sizeof(cx<T>);
    static constexpr size_t fixed = 128 + x_bytes + ytw_bytes;
    static constexpr int NB = fixed + 3 * tile_bytes <= 227 * 1024 ? 3 : 2;  // y tile ring
    static constexpr size_t smem = fixed + NB * tile_bytes;
};

// ------------------------------------------------------------------------------------------------------------------
// forward: X group.  Real rows -> half spectrum rows of the ring plane (tiled [g][y][L]); the row transform is the one
// of k2_xfwd (fe_fft2_x.cu): complex transform of length MX on z[j] = x[2j] + i x[2j+1], then the split step.
// ------------------------------------------------------------------------------------------------------------------
template <typename T, int MX, int MY>
__device__ __forceinline__ void xy_fwd_xgroup(const T* __restrict__ in, cx<T>* ring, const XYArgs& a, unsigned char* smem, int t)
{
    using C = XYCfg<T, MX, MY>;
    constexpr int R1 = C::R1, R2 = C::R2, TPP = R2, NT3 = R1 / TPP, ROWS = C::ROWS;
    constexpr int L = C::LANES;
    cx<T>* tw = reinterpret_cast<cx<T>*>(smem);       // w_MX^(n2 k1) at [k1 * R2 + n2]
    cx<T>* tws = tw + MX;                             // w_2MX^k
    cx<T>* buf = tws + MX;
    const int tp = t % TPP, rl = t / TPP;
    cx<T>* rb = buf + rl * C::RPITCH;
    constexpr int NLOAD = R1 / 2;                     // zero-padded axis: the upper half of the input is zero
    const int ntasks = a.nplanes * a.xgroups;
    auto fetch = [&](int q, cx<T>* dst) {
        if (q < ntasks) {
            const int p = q / a.xgroups, rg = q - p * a.xgroups;
            const int64_t row = (int64_t)p * a.ny + rg * ROWS + rl;
            const cx<T>* src = reinterpret_cast<const cx<T>*>(in + row * a.real_rs) + tp;
            static_for<NLOAD>([&](auto ic) {
                constexpr int n1 = decltype(ic)::value;
                dst[n1] = (tp + R2 * n1 < a.nc) ? src[R2 * n1] : cx<T>{0, 0};
            });
        } else {
            static_for<NLOAD>([&](auto ic) { dst[decltype(ic)::value] = cx<T>{0, 0}; });
        }
    };
    cx<T> vn[NLOAD];
    fetch(blockIdx.x, vn);
    {
        const cx<T>* twg = static_cast<const cx<T>*>(a.tw);
        for (int e = t; e < MX; e += 256) {
            tw[e] = twg[((e / R2) * (e % R2)) * (kTwiddleN / MX)];
            tws[e] = twg[e * (kTwiddleN / (2 * MX))];
        }
    }
    xy_bar(1);
    for (int q = blockIdx.x; q < ntasks; q += gridDim.x) {
        const int p = q / a.xgroups, rg = q - p * a.xgroups;
        cx<T> v[R1];
        static_for<NLOAD>([&](auto ic) { v[decltype(ic)::value] = vn[decltype(ic)::value]; });
        fetch(q + gridDim.x, vn);
        Dif<T, -1, R1, 0, true>::run(v);
        static_for<R1>([&](auto pc) {
            constexpr int pp = decltype(pc)::value;
            constexpr int k1 = brev<R1>(pp);
            cx<T> val = v[pp];
            if constexpr (k1 != 0) val = cmul(val, tw[k1 * R2 + tp]);
            rb[k1 * (R2 + 1) + tp] = val;
        });
        xy_bar(1);
        cx<T> u[NT3][R2];
#pragma unroll
        for (int it = 0; it < NT3; ++it) {
            const int k1 = tp + it * TPP;
            static_for<R2>([&](auto nc) { u[it][decltype(nc)::value] = rb[k1 * (R2 + 1) + decltype(nc)::value]; });
            Dif<T, -1, R2>::run(u[it]);
        }
        xy_bar(1);
#pragma unroll
        for (int it = 0; it < NT3; ++it) {
            const int k1 = tp + it * TPP;
            static_for<R2>([&](auto pc) {
                constexpr int pp = decltype(pc)::value;
                rb[k1 + R1 * brev<R2>(pp)] = u[it][pp];
            });
        }
        // the ring slot of this plane is free once every tile of plane p - ring has been read
        if (t == 0 && p >= a.ring) xy_wait(a.ydone + (p - a.ring), a.G, a.err);
        xy_bar(1);
        {
            const int y = rg * ROWS + rl;
            cx<T>* dst = ring + (int64_t)(p % a.ring) * a.ring_plane + (int64_t)y * L;
            const int64_t sg = (int64_t)a.ny * L;
            for (int k = tp; k <= MX / 2; k += TPP) {
                const cx<T> Zk = rb[k], Zn = rb[(MX - k) & (MX - 1)];
                const T ex = (T)0.5 * (Zk.x + Zn.x), ey = (T)0.5 * (Zk.y - Zn.y);
                const T ox = (T)0.5 * (Zk.y + Zn.y), oy = (T)-0.5 * (Zk.x - Zn.x);
                const cx<T> w = tws[k];
                const T px = ox * w.x - oy * w.y, py = ox * w.y + oy * w.x;
                const int k2 = MX - k;
                dst[(int64_t)(k >> a.lg) * sg + (k & (L - 1))] = {ex + px, ey + py};
                dst[(int64_t)(k2 >> a.lg) * sg + (k2 & (L - 1))] = {ex - px, py - ey};
            }
        }
        xy_fence_proxy();                 // these generic-proxy stores are read by bulk copies (async proxy)
        xy_bar(1);                        // all rows of the task stored; row buffer free for the next task
        if (t == 0) {
            __threadfence();
            xy_red_release(a.xdone + p);
        }
    }
}

// ------------------------------------------------------------------------------------------------------------------
// Three-level in-place transform of one y tile in shared memory (the scheme of k4_axis, fe_fft2_axis.cu):
//   MY = RA RB RC, n = n3 + RC n2 + RC RB n1, k = k1 + RA k2 + RA RB k3;
//   forward: rows y (first half data, rest zero) in, frequency k at slot (k1 RB + k2) RC + k3 out ("slot order");
//   inverse: slot order in, rows y out (first half kept).
// `after_first` runs between the first and the second level (the caller issues the next tile's load there).
// ------------------------------------------------------------------------------------------------------------------
template <typename T, int MY, int DIR, typename F>
__device__ __forceinline__ void xy_tile_transform(cx<T>* buf /* + lane */, const cx<T>* tw, int tp, F&& after_first)
{
    constexpr int RA = XYFact3<MY>::RA, RB = XYFact3<MY>::RB, RC = XYFact3<MY>::RC;
    constexpr int LANES = 128 / (int)sizeof(cx<T>);
    constexpr int TPP = 256 / LANES;
    constexpr int NTA = RB * RC, NTB = RA * RC, NTC = RA * RB;
    static_assert(NTA % TPP == 0 && NTB % TPP == 0 && NTC % TPP == 0, "tasks must divide evenly");
    if (DIR < 0) {
#pragma unroll
        for (int it = 0; it < NTA / TPP; ++it) {
            const int j = tp + it * TPP;
            cx<T> u[RA];
            cx<T>* col = buf + j * LANES;
            static_for<RA / 2>([&](auto ic) { u[decltype(ic)::value] = col[decltype(ic)::value * RB * RC * LANES]; });
            cx<T> w[RA];
            static_for<RA - 1>([&](auto kc) { w[decltype(kc)::value + 1] = tw[j * (decltype(kc)::value + 1)]; });
            Dif<T, DIR, RA, 0, true>::run(u);
            static_for<RA>([&](auto pc) {
                constexpr int p = decltype(pc)::value;
                constexpr int k1 = brev<RA>(p);
                cx<T> val = u[p];
                if constexpr (k1 != 0) val = cmul(val, w[k1]);
                col[k1 * RB * RC * LANES] = val;
            });
        }
        xy_bar(2);
        after_first();
#pragma unroll
        for (int it = 0; it < NTB / TPP; ++it) {
            const int tb = tp + it * TPP, n3 = tb % RC, k1 = tb / RC;
            cx<T> u[RB];
            cx<T>* col = buf + (k1 * RB * RC + n3) * LANES;
            static_for<RB>([&](auto nc) { u[decltype(nc)::value] = col[decltype(nc)::value * RC * LANES]; });
            cx<T> w[RB];
            static_for<RB - 1>([&](auto kc) { w[decltype(kc)::value + 1] = tw[RA * n3 * (decltype(kc)::value + 1)]; });
            Dif<T, DIR, RB>::run(u);
            static_for<RB>([&](auto pc) {
                constexpr int p = decltype(pc)::value;
                constexpr int k2 = brev<RB>(p);
                cx<T> val = u[p];
                if constexpr (k2 != 0) val = cmul(val, w[k2]);
                col[k2 * RC * LANES] = val;
            });
        }
        xy_bar(2);
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
#pragma unroll
        for (int it = 0; it < NTC / TPP; ++it) {
            const int tc = tp + it * TPP, k2 = tc % RB;
            cx<T> u[RC];
            cx<T>* col = buf + tc * RC * LANES;
            static_for<RC>([&](auto nc) { u[decltype(nc)::value] = col[decltype(nc)::value * LANES]; });
            cx<T> w[RC];
            static_for<RC - 1>([&](auto nc) { w[decltype(nc)::value + 1] = tw[RA * (decltype(nc)::value + 1) * k2]; });
            Dif<T, DIR, RC>::run(u);
            static_for<RC>([&](auto pc) {
                constexpr int p = decltype(pc)::value;
                constexpr int n3 = brev<RC>(p);
                cx<T> val = u[p];
                if constexpr (n3 != 0) val = cmulc(val, w[n3]);
                col[n3 * LANES] = val;
            });
        }
        xy_bar(2);
        after_first();
#pragma unroll
        for (int it = 0; it < NTB / TPP; ++it) {
            const int tb = tp + it * TPP, n3 = tb % RC, k1 = tb / RC;
            cx<T> u[RB];
            cx<T>* col = buf + (k1 * RB * RC + n3) * LANES;
            static_for<RB>([&](auto nc) { u[decltype(nc)::value] = col[decltype(nc)::value * RC * LANES]; });
            cx<T> w[RB];
            static_for<RB>([&](auto nc) { w[decltype(nc)::value] = tw[(n3 + RC * decltype(nc)::value) * k1]; });
            Dif<T, DIR, RB>::run(u);
            static_for<RB>([&](auto pc) {
                constexpr int p = decltype(pc)::value;
                constexpr int n2 = brev<RB>(p);
                col[n2 * RC * LANES] = cmulc(u[p], w[n2]);
            });
        }
        xy_bar(2);
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
                if constexpr (n1 < RA / 2) col[n1 * RB * RC * LANES] = u[p];
            });
        }
    }
}

// forward: Y group.  Tile j = (plane p, kx group g) in plane-major order; tiles of a block are j = blockIdx.x + i gridDim.x.
template <typename T, int MX, int MY>
__device__ __forceinline__ void xy_fwd_ygroup(const cx<T>* ring, cx<T>* S2, const XYArgs& a, unsigned long long* bars,
                                              cx<T>* tw, cx<T>* bufs, int t)
{
    using C = XYCfg<T, MX, MY>;
    constexpr int NB = C::NB, TILE = C::TILE, LANES = C::LANES;
    const int lane = t % LANES, tp = t / LANES;
    const unsigned in_bytes = (unsigned)(a.ny * LANES * sizeof(cx<T>));
    const unsigned out_bytes = (unsigned)(MY * LANES * sizeof(cx<T>));
    const int ntiles = a.nplanes * a.G;
    if (t == 0) {
        for (int b = 0; b < NB; ++b) xy_mbar_init(&bars[b], 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    load_twiddles<T, MY>(tw, static_cast<const cx<T>*>(a.tw), t, 256);
    xy_bar(2);
    // thread 0: wait for the rows of the tile's plane, then start the bulk copy of the tile
    auto issue = [&](int j, int b) {
        if (j >= ntiles) return;
        const int p = j / a.G, g = j - p * a.G;
        xy_wait(a.xdone + p, a.xgroups, a.err);
        xy_fence_proxy();
        xy_mbar_expect_tx(&bars[b], in_bytes);
        xy_bulk_load(bufs + b * TILE, ring + (int64_t)(p % a.ring) * a.ring_plane + (int64_t)g * a.ny * LANES, in_bytes, &bars[b]);
    };
    if (t == 0) {
#pragma unroll
        for (int pre = 0; pre < NB - 1; ++pre) issue(blockIdx.x + pre * gridDim.x, pre);
    }
    int i = 0;
    for (int j = blockIdx.x; j < ntiles; j += gridDim.x, ++i) {
        const int b = i % NB;
        const int p = j / a.G, g = j - p * a.G;
        xy_mbar_wait(&bars[b], (unsigned)((i / NB) & 1));
        if (t == 0) xy_red_release(a.ydone + p);             // the tile has left the ring
        xy_tile_transform<T, MY, -1>(bufs + b * TILE + lane, tw, tp, [&]() {
            if (t == 0) {
                xy_bulk_wait_read<0>();                      // the store of tile i-1 has released its buffer
                issue(j + (NB - 1) * gridDim.x, (i + NB - 1) % NB);
            }
        });
        xy_fence_async_smem();
        xy_bar(2);
        if (t == 0) {
            const int bc = p / a.nz, z = p - bc * a.nz;
            xy_bulk_store(S2 + (int64_t)bc * a.s2_sb + (int64_t)z * a.s2_sz + (int64_t)g * a.s2_sg, bufs + b * TILE, out_bytes);
        }
    }
    if (t == 0) xy_bulk_wait_read<0>();
}

template <typename T, int MX, int MY>
__global__ void __launch_bounds__(512, 1) k_xyfwd(const T* __restrict__ P, cx<T>* ring, cx<T>* S2, XYArgs a)
{
    using C = XYCfg<T, MX, MY>;
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(fe2_smem);
    unsigned char* xs = fe2_smem + 128;
    cx<T>* ytw = reinterpret_cast<cx<T>*>(xs + C::x_bytes);
    cx<T>* bufs = ytw + MY;
    if (threadIdx.x < 256) xy_fwd_xgroup<T, MX, MY>(P, ring, a, xs, (int)threadIdx.x);
    else xy_fwd_ygroup<T, MX, MY>(ring, S2, a, bars, ytw, bufs, (int)threadIdx.x - 256);
}

template <typename T, int MX, int MY>
static cudaError_t launch_xyfwd_one(const T* P, void* ring, void* S2, XYArgs a, cudaStream_t st)
{
    using C = XYCfg<T, MX, MY>;
    static PerDevice<int> cache;
    int& nblocks = cache.here();
    if (!nblocks) {
        cudaError_t e = cudaFuncSetAttribute(k_xyfwd<T, MX, MY>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem);
        if (e != cudaSuccess) return e;
        int dev = 0, sms = 0, per = 0;
        if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, k_xyfwd<T, MX, MY>, 512, C::smem)) != cudaSuccess) return e;
        if (per < 1) return cudaErrorLaunchOutOfResources;
        nblocks = sms;
    }
    a.xgroups = a.ny / C::ROWS;
    const int ntiles = a.nplanes * a.G;
    const int grid = ntiles < nblocks ? ntiles : nblocks;
    cx<T>* ringp = static_cast<cx<T>*>(ring);
    cx<T>* s2p = static_cast<cx<T>*>(S2);
    void* args[] = {(void*)&P, (void*)&ringp, (void*)&s2p, (void*)&a};
    return cudaLaunchCooperativeKernel((const void*)k_xyfwd<T, MX, MY>, dim3(grid), dim3(512), args, C::smem, st);
}

}  // namespace v2

// planes a ring can hold without leaving L2, and the rows-per-task constraint
bool xy_supported(int Mx, int My, int nx, int ny)
{
    if (!(Mx == 128 || Mx == 256) || !(My == 256 || My == 512)) return false;
    if (2 * ny != My || nx > Mx || (nx & 1)) return false;      // both axes zero-padded, full first half of y
    const int rows = Mx == 256 ? 16 : 32;
    return ny % rows == 0;
}

template <typename T>
cudaError_t launch_xyfwd(const FftCtx& c, const T* P, void* ring, void* S2, int nx, int ny, int nz, int nplanes, int G,
                         int ring_slots, int64_t s2_sz, int64_t s2_sg, int64_t s2_sb, int* counters, cudaStream_t st)
{
    const int Mx = c.plan[0].M, My = c.plan[1].M;
    if (!xy_supported(Mx, My, nx, ny) || ring_slots < 2) return cudaErrorInvalidValue;
    constexpr int L = 128 / (int)sizeof(v2::cx<T>);
    int lg = 0;
    while ((1 << lg) < L) ++lg;
    cudaError_t e = cudaMemsetAsync(counters, 0, (size_t)(2 * nplanes + 1) * sizeof(int), st);
    if (e != cudaSuccess) return e;
    v2::XYArgs a{c.tw, nplanes, nz, ny, G, ring_slots, nx / 2, lg, 0, nx, (int64_t)G * ny * L, s2_sz, s2_sg, s2_sb,
                 counters, counters + nplanes, counters + 2 * nplanes};
    if (Mx == 256 && My == 512) return v2::launch_xyfwd_one<T, 256, 512>(P, ring, S2, a, st);
    if (Mx == 128 && My == 256) return v2::launch_xyfwd_one<T, 128, 256>(P, ring, S2, a, st);
    if (Mx == 256 && My == 256) return v2::launch_xyfwd_one<T, 256, 256>(P, ring, S2, a, st);
    if (Mx == 128 && My == 512) return v2::launch_xyfwd_one<T, 128, 512>(P, ring, S2, a, st);
    return cudaErrorInvalidValue;
}

template cudaError_t launch_xyfwd<double>(const FftCtx&, const double*, void*, void*, int, int, int, int, int, int, int64_t,
                                          int64_t, int64_t, int*, cudaStream_t);
template cudaError_t launch_xyfwd<float>(const FftCtx&, const float*, void*, void*, int, int, int, int, int, int, int64_t,
                                         int64_t, int64_t, int*, cudaStream_t);

}  // namespace fe
