// fe_fft2_z.cu -- size-specialised fused z pass (Eq. 5-6 in k-space):
// forward z transform of the three components, E~_i = -escale * sum_j K~_ij P~_j, inverse z transform, in place
// on S[b][3][nz][My][pitch].  K~ is real and symmetric, stored for kz <= Mz/2, ky <= My/2; the odd components
// change sign under ky -> -ky (xy, yz) and kz -> -kz (xz, yz).
//
// Persistent blocks, software pipelined with cp.async:
//   work item  = (group of LANES consecutive kx, |ky|): the K~ tile of the item is copied to shared memory once and
//                serves the tiles ky, My - ky of every batch member;
//   tile       = LANES pencils x 3 components; its nz input rows are prefetched into a staging buffer while the
//                previous tile is being transformed.
// Per tile, one thread holds the spectrum of all three components at the R2 frequencies kz = k1 + R1 k2 in
// registers, so the multiply and the first stage of the inverse transform need no shared-memory round trip:
//   forward   x[n2 + R2 n1] -> (R1-point over n1) -> exchange -> twiddle -> (R2-point over n2) -> X[k1 + R1 k2]
//   inverse   X[k1 + R1 k2] -> (R2-point over k2) -> twiddle -> exchange -> (R1-point over k1) -> x[n1 R2 + n2]
// Both inter-step twiddles w_M^{+-n2 k1} are applied by the thread that owns k1: it loads its R2 - 1 factors once
// per tile and uses them for the three components in both directions (the R1-point steps move no twiddles).
#include "fe_fft2.cuh"
#include <string.h>
#include <cuda.h>          // CUtensorMap and cuTensorMapEncodeTiled's signature only; the entry point is fetched at run time

namespace fe {
namespace v2 {

// ---- tensor-copy (TMA) staging of the tiled layouts: one copy per tile / per K~ tile, completion on an mbarrier ----------
__device__ __forceinline__ unsigned z_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void z_mbar_init(void* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(z_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void z_mbar_expect_tx(void* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(z_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void z_mbar_wait(void* bar, unsigned parity)
{
    const unsigned addr = z_smem_u32(bar);
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
__device__ __forceinline__ void z_tma_load_5d(void* smem_dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, int c4, void* bar)
{
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5, %6}], [%7];\n" ::"r"(
            z_smem_u32(smem_dst)),
        "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(z_smem_u32(bar))
        : "memory");
}

// factorisation used by the fused pass: R2 frequencies per thread (3 components in registers)
template <int M> struct ZFact;
template <> struct ZFact<64> { static constexpr int R1 = 8, R2 = 8; };
template <> struct ZFact<128> { static constexpr int R1 = 16, R2 = 8; };
template <> struct ZFact<256> { static constexpr int R1 = 32, R2 = 8; };

// Spectrum element (b, c, z, ky, kx) sits at b * 3 * cs + c * cs + z * s_z + ky * s_ky + (kx / LANES) * s_g + kx % LANES,
// tensor element (c6, kz, ky, kx) at c6 * kcs + kz * k_skz + ky * k_sky + (kx / LANES) * k_sg + kx % LANES
// (complex / real elements), which covers the row-major and the tiled layouts of fe_api.cu.
struct Z2Args {
    const void* tw;
    const DevMember* members;
    int My, batch, nz;         // nz: data rows per pencil (<= M/2 on a zero-padded axis)
    int ngroups;      // groups of LANES consecutive kx
    int nitems;       // ngroups * (My/2 + 1)
    int64_t cs, s_z, s_ky, s_g;
    int64_t kcs, k_skz, k_sky, k_sg;
    int la, lb, lc;   // ky is stored in slot order (k1 pb + k2) pc + k3, ky = k1 + pa k2 + pa pb k3, with the binary
                      // logarithms of pa, pb, pc given; la < 0: natural order
};

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(s), "l"(gmem));
}
// copy BYTES (8 or 16) bytes
template <int BYTES> __device__ __forceinline__ void cp_async_n(void* smem, const void* gmem)
{
    if constexpr (BYTES == 16) cp_async16(smem, gmem);
    else cp_async8(smem, gmem);
}
// x with its sign bit flipped when s = 0x80000000 (integer pipe: keeps the sign changes of the odd tensor
// components out of the floating-point pipe)
__device__ __forceinline__ double xorsign(double x, unsigned s)
{
    return __hiloint2double(__double2hiint(x) ^ (int)s, __double2loint(x));
}
__device__ __forceinline__ float xorsign(float x, unsigned s) { return __uint_as_float(__float_as_uint(x) ^ s); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

template <typename T, int M, int LANES, bool PRUNE> struct ZCfg {
    static constexpr int R1 = ZFact<M>::R1, R2 = ZFact<M>::R2;
    static constexpr int TPP = R1;                          // threads per pencil (one step-3 task each)
    static constexpr int THREADS = LANES * TPP;
    static constexpr int NT1 = (3 * R2 + TPP - 1) / TPP;    // step-1 tasks (component, n2) per thread
    // exchange tile of one component: rows of LANES complex.  When a row is shorter than 128 bytes two threads
    // of one shared-memory phase sit in rows R2 (forward) or R1 (inverse) apart; one pad row per group of R2 / R1
    // rows shifts them into different bank halves.
    static constexpr int PAD = LANES * (int)sizeof(cx<T>) < 128 ? 1 : 0;
    static constexpr int P2 = R2 + PAD, P1 = R1 + PAD;      // row pitch of a k1 group (forward) / n2 group (inverse)
    static constexpr int TILE = (R1 * P2 > R2 * P1 ? R1 * P2 : R2 * P1) * LANES;
    static constexpr int NIN = PRUNE ? M / 2 : M;           // input rows per component
    static constexpr int HZ = M / 2 + 1;
    static constexpr size_t tw_bytes = (size_t)M * sizeof(cx<T>);
    static constexpr size_t ex_bytes = (size_t)3 * TILE * sizeof(cx<T>);
    static constexpr size_t st_bytes = (size_t)3 * NIN * LANES * sizeof(cx<T>);
    static constexpr size_t k_bytes = ((size_t)6 * HZ * LANES * sizeof(T) + 15) / 16 * 16;
    static constexpr size_t smem = tw_bytes + ex_bytes + st_bytes + k_bytes + 16;       // + two mbarriers (TMA staging)
};

// position of a block in its sequence of tiles; advanced without divisions (the loop head is executed by every
// thread once per tile, and its integer chain is not hidden by anything else)
struct ZIter {
    int kxg, kyh;             // work item
    int b, m, nm;             // batch member, mirror index (ky = m ? My - kyh : kyh), mirrors of the item (1 or 2)
    __device__ __forceinline__ void set_item(int g, int h, const Z2Args& a)
    {
        kxg = g;
        kyh = h;
        b = 0;
        m = 0;
        nm = (h == 0 || 2 * h == a.My) ? 1 : 2;
    }
    __device__ __forceinline__ bool valid(const Z2Args& a) const { return 2 * kyh <= a.My; }
    // dq, dr: quotient and remainder of gridDim.x by a.ngroups
    __device__ __forceinline__ void next(const Z2Args& a, int dq, int dr)
    {
        if (++m < nm) return;
        m = 0;
        if (++b < a.batch) return;
        int g = kxg + dr, h = kyh + dq;
        if (g >= a.ngroups) {
            g -= a.ngroups;
            ++h;
        }
        set_item(g, h, a);
    }
    __device__ __forceinline__ bool same_item(const ZIter& o) const { return kxg == o.kxg && kyh == o.kyh; }
    __device__ __forceinline__ int ky(const Z2Args& a) const { return m ? a.My - kyh : kyh; }
};

// TMA = true (tiled layouts): the rows of a tile (box LANES x 1 ky x NIN rows x 1 kx group x 3 components of S) and the
// K~ tile of an item (box LANES x HZ x 1 x 1 x 6 of Kt) each arrive as ONE tensor copy issued by thread 0 and completed on
// an mbarrier, instead of 12 + 9 cp.async per thread and tile; rows beyond nz are zero-filled by the copy engine.
template <typename T, int M, int LANES, bool PRUNE, bool TMA = false>
__global__ void __launch_bounds__(ZCfg<T, M, LANES, PRUNE>::THREADS, ZCfg<T, M, LANES, PRUNE>::THREADS <= 64 ? 4 : (ZCfg<T, M, LANES, PRUNE>::smem > 112 * 1024 ? 1 : 2))
k2_zmul(cx<T>* __restrict__ S, const T* __restrict__ Kt, Z2Args a, const __grid_constant__ CUtensorMap smap,
        const __grid_constant__ CUtensorMap kmap)
{
    using C = ZCfg<T, M, LANES, PRUNE>;
    constexpr int R1 = C::R1, R2 = C::R2, TPP = C::TPP, NT1 = C::NT1, TILE = C::TILE, NIN = C::NIN, HZ = C::HZ;
    constexpr int P1 = C::P1, P2 = C::P2;
    cx<T>* tw = reinterpret_cast<cx<T>*>(fe2_smem);
    cx<T>* buf = tw + M;                                            // exchange [3][M][LANES]
    cx<T>* stage = buf + 3 * TILE;                                  // staged input [3][NIN][LANES]
    T* kbuf = reinterpret_cast<T*>(stage + 3 * NIN * LANES);        // K~ tile [6][HZ][LANES]
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(reinterpret_cast<unsigned char*>(kbuf) + C::k_bytes);  // [2]
    const int lane = threadIdx.x % LANES, tp = threadIdx.x / LANES;
    const int64_t sa = a.s_z, cs = a.cs, kcs = a.kcs;

    auto tile_base = [&](const ZIter& it) -> cx<T>* {
        const int ky = it.ky(a);
        int slot = ky;
        if (a.la >= 0)
            slot = ((ky & ((1 << a.la) - 1)) << (a.lb + a.lc)) | (((ky >> a.la) & ((1 << a.lb) - 1)) << a.lc) |
                   (ky >> (a.la + a.lb));
        return S + (int64_t)it.b * 3 * cs + (int64_t)slot * a.s_ky + (int64_t)it.kxg * a.s_g;
    };
    // asynchronous copies: input rows of a tile, K~ tile of an item
    auto prefetch_tile = [&](const cx<T>* tb) {
        constexpr int CB = LANES * (int)sizeof(cx<T>) < 16 ? 8 : 16;   // bytes per copy
        constexpr int PER = CB / (int)sizeof(cx<T>);                    // complex elements per copy
        constexpr int OPS_ROW = LANES / PER;                            // copies per row
        constexpr int RSTEP = C::THREADS / OPS_ROW;                     // rows covered by one sweep of the block
        static_assert(C::THREADS % OPS_ROW == 0 && NIN % RSTEP == 0, "tile copy must be regular");
        const int q = threadIdx.x % OPS_ROW, row0 = threadIdx.x / OPS_ROW;
        const cx<T>* g = tb + (int64_t)row0 * sa + q * PER;
        cx<T>* s = stage + row0 * LANES + q * PER;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
#pragma unroll
            for (int j = 0; j < NIN / RSTEP; ++j)
                if (!PRUNE || row0 + j * RSTEP < a.nz)          // rows nz .. M/2 of a zero-padded axis stay zero
                    cp_async_n<CB>(s + (c * NIN + j * RSTEP) * LANES, g + c * cs + (int64_t)(j * RSTEP) * sa);
        }
    };
    // K~ tile of an item, copied by the NTH threads [T0, T0 + NTH) of the block
    auto prefetch_k = [&](const ZIter& it, auto nth_c, auto t0_c) {
        constexpr int NTH = decltype(nth_c)::value, T0 = decltype(t0_c)::value;
        constexpr int CB = LANES * (int)sizeof(T) < 16 ? 8 : 16;
        constexpr int PER = CB / (int)sizeof(T);
        constexpr int OPS_ROW = LANES / PER;
        constexpr int RSTEP = NTH / OPS_ROW;
        static_assert(LANES * sizeof(T) >= 8 && NTH % OPS_ROW == 0, "a K~ row of a tile must be at least 8 bytes");
        const int tid = (int)threadIdx.x - T0;
        const int q = tid % OPS_ROW, row0 = tid / OPS_ROW;
        const int64_t krs = a.k_skz;                                    // stride of kz in the table
        const T* g = Kt + (int64_t)it.kyh * a.k_sky + (int64_t)it.kxg * a.k_sg + (int64_t)row0 * krs + q * PER;
        T* s = kbuf + row0 * LANES + q * PER;
#pragma unroll
        for (int c6 = 0; c6 < 6; ++c6) {
#pragma unroll
            for (int j = 0; j < (HZ + RSTEP - 1) / RSTEP; ++j)
                if ((j + 1) * RSTEP <= HZ || row0 + j * RSTEP < HZ)
                    cp_async_n<CB>(s + (c6 * HZ + j * RSTEP) * LANES, g + c6 * kcs + (int64_t)(j * RSTEP) * krs);
        }
    };
    using ic_all = std::integral_constant<int, C::THREADS>;
    using ic_zero = std::integral_constant<int, 0>;
    // threads without a task in the R1-point steps (TPP > 3 R2): they fetch the next K~ tile during inverse step 2
    constexpr int NIDLE = NT1 == 1 && 3 * R2 < TPP ? (TPP - 3 * R2) * LANES : 0;

    ZIter cur;
    cur.set_item(blockIdx.x % a.ngroups, blockIdx.x / a.ngroups, a);
    if (!cur.valid(a)) return;
    const int dq = gridDim.x / a.ngroups, dr = gridDim.x % a.ngroups;
    // tensor-copy staging: thread 0 issues, everybody waits on the mbarriers (bars[0]: tile rows, bars[1]: K~ tile)
    auto tma_tile = [&](const ZIter& it) {
        const int ky = it.ky(a);
        int slot = ky;
        if (a.la >= 0)
            slot = ((ky & ((1 << a.la) - 1)) << (a.lb + a.lc)) | (((ky >> a.la) & ((1 << a.lb) - 1)) << a.lc) |
                   (ky >> (a.la + a.lb));
        z_mbar_expect_tx(&bars[0], (unsigned)(3 * NIN * LANES * sizeof(cx<T>)));
        z_tma_load_5d(stage, &smap, 0, slot, 0, it.kxg, 3 * it.b, &bars[0]);
    };
    auto tma_k = [&](const ZIter& it) {
        z_mbar_expect_tx(&bars[1], (unsigned)(6 * HZ * LANES * sizeof(T)));
        z_tma_load_5d(kbuf, &kmap, 0, 0, it.kyh, it.kxg, 0, &bars[1]);
    };
    unsigned sphase = 0, kphase = 0;
    bool kpend = true;
    if (!TMA && PRUNE && a.nz < NIN) {      // padding rows inside the staged half: cleared once, never written again
        for (int e = threadIdx.x; e < 3 * NIN * LANES; e += C::THREADS) stage[e] = cx<T>{0, 0};
        __syncthreads();
    }
    cx<T>* cur_base = tile_base(cur);       // carried from the prefetch of a tile to its turn in the loop
    if (TMA) {
        if (threadIdx.x == 0) {
            z_mbar_init(&bars[0], 1);
            z_mbar_init(&bars[1], 1);
            asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
            tma_tile(cur);
            tma_k(cur);
        }
    } else {
        prefetch_tile(cur_base);
        cp_async_commit();                  // group A: input of the first tile
        prefetch_k(cur, ic_all{}, ic_zero{});
        cp_async_commit();                  // group B: K~ of the first item
    }
    load_twiddles<T, M>(tw, static_cast<const cx<T>*>(a.tw), threadIdx.x, C::THREADS);

    while (cur.valid(a)) {
        const int ky = cur.ky(a);
        cx<T>* base = cur_base + lane;
        const double escale = a.members[cur.b].escale;  // issued here, consumed after the forward transform
        ZIter nxt = cur;
        nxt.next(a, dq, dr);
        if (TMA) {
            __syncthreads();                // (first tile: mbarriers initialised) previous tile's exchange reads are done
            z_mbar_wait(&bars[0], sphase);  // this tile's input has landed
            sphase ^= 1;
        } else {
            cp_async_wait<1>();             // this tile's input has landed (the newest group may still be in flight)
            __syncthreads();                // ... for every thread; also: previous tile's exchange reads are done
        }
        // ---- forward step 1: tasks (c, n2): R1-point over n1 (inputs in bit-reversed register order, k1 natural)
#pragma unroll
        for (int it = 0; it < NT1; ++it) {
            const int task = tp + it * TPP;
            if ((3 * R2) % TPP == 0 || task < 3 * R2) {
                const int c = task / R2, n2 = task % R2;
                cx<T> w[R1];
                const cx<T>* src = stage + (c * NIN + n2) * LANES + lane;
                static_for<R1>([&](auto pc) {
                    constexpr int p = decltype(pc)::value;
                    constexpr int n1 = brev<R1>(p);
                    if constexpr (!PRUNE || n1 < R1 / 2) w[p] = src[n1 * R2 * LANES];
                });
                DitF<T, -1, R1, 0, PRUNE, false>::run(w);
                cx<T>* dst = buf + c * TILE + n2 * LANES + lane;
                static_for<R1>([&](auto kc) { dst[decltype(kc)::value * P2 * LANES] = w[decltype(kc)::value]; });
            }
        }
        __syncthreads();                    // exchange written, staging buffer free
        if (nxt.valid(a)) {
            cur_base = tile_base(nxt);
            if (TMA) { if (threadIdx.x == 0) tma_tile(nxt); }
            else prefetch_tile(cur_base);
        }
        if (!TMA) cp_async_commit();        // group A (possibly empty): input of the next tile
        // ---- forward step 3 for thread k1 = tp: twiddle, R2-point over n2; u[c][p] = P~_c[k1 + R1 brev(p)]
        const int k1 = tp;
        cx<T> wk[R2];                       // w_M^{n2 k1}, n2 = 1 .. R2-1 (wk[0] unused)
        static_for<R2 - 1>([&](auto nc) { wk[decltype(nc)::value + 1] = tw[(decltype(nc)::value + 1) * k1]; });
        cx<T> u[3][R2];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const cx<T>* src = buf + c * TILE + k1 * P2 * LANES + lane;
            static_for<R2>([&](auto nc) { u[c][decltype(nc)::value] = src[decltype(nc)::value * LANES]; });
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            static_for<R2 - 1>([&](auto nc) {
                constexpr int n2 = decltype(nc)::value + 1;
                u[c][n2] = cmul(u[c][n2], wk[n2]);
            });
            Dif<T, -1, R2>::run(u[c]);
        }
        if (TMA) {
            if (kpend) {                    // K~ of this item has landed
                z_mbar_wait(&bars[1], kphase);
                kphase ^= 1;
                kpend = false;
            }
        } else {
            cp_async_wait<1>();             // K~ of this item has landed (only the group just committed may be pending)
        }
        __syncthreads();                    // ... for every thread; exchange fully read
        // ---- multiply
        {
            const unsigned sy = 2 * ky > a.My ? 0x80000000u : 0u;      // sign bits of the odd components
            static_for<R2>([&](auto pc) {
                constexpr int p = decltype(pc)::value;
                constexpr int k2 = brev<R2>(p);
                const int kz = k1 + R1 * k2;
                const int kzm = 2 * kz <= M ? kz : M - kz;
                const unsigned sz = 2 * kz > M ? 0x80000000u : 0u;
                const T* kp = kbuf + kzm * LANES + lane;
                const T Kxx = kp[0], Kyy = kp[HZ * LANES], Kzz = kp[2 * HZ * LANES];
                const T Kxy = xorsign(kp[3 * HZ * LANES], sy), Kxz = xorsign(kp[4 * HZ * LANES], sz);
                const T Kyz = xorsign(kp[5 * HZ * LANES], sy ^ sz);
                const cx<T> Px = u[0][p], Py = u[1][p], Pz = u[2][p];
                u[0][p] = {Kxx * Px.x + Kxy * Py.x + Kxz * Pz.x, Kxx * Px.y + Kxy * Py.y + Kxz * Pz.y};
                u[1][p] = {Kxy * Px.x + Kyy * Py.x + Kyz * Pz.x, Kxy * Px.y + Kyy * Py.y + Kyz * Pz.y};
                u[2][p] = {Kxz * Px.x + Kyz * Py.x + Kzz * Pz.x, Kxz * Px.y + Kyz * Py.y + Kzz * Pz.y};
            });
        }
        // ---- inverse step 1: R2-point over k2 (bit-reversed in, natural n2 out), twiddle, exchange.  The factor
        // -escale of Eq. 6 rides on the twiddles (2 (R2 - 1) + 6 multiplications instead of 6 R2 on the tensor).
        {
            const T esc = (T)(-escale);
            static_for<R2 - 1>([&](auto nc) {
                constexpr int n2 = decltype(nc)::value + 1;
                wk[n2] = {esc * wk[n2].x, esc * wk[n2].y};
            });
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                DitF<T, +1, R2>::run(u[c]);
                cx<T>* dst = buf + c * TILE + k1 * LANES + lane;
                static_for<R2>([&](auto nc) {
                    constexpr int n2 = decltype(nc)::value;
                    cx<T> val = u[c][n2];
                    if constexpr (n2 != 0) val = cmulc(val, wk[n2]);
                    else val = {esc * val.x, esc * val.y};
                    dst[n2 * P1 * LANES] = val;
                });
            }
        }
        __syncthreads();                    // exchange written; every thread is past the multiply: K~ buffer free
        if (TMA) {
            if (nxt.valid(a) && !nxt.same_item(cur)) {
                if (threadIdx.x == 0) tma_k(nxt);
                kpend = true;
            }
        } else if (nxt.valid(a) && !nxt.same_item(cur)) {
            if constexpr (NIDLE > 0) {
                if (tp >= 3 * R2)
                    prefetch_k(nxt, std::integral_constant<int, NIDLE>{}, std::integral_constant<int, 3 * R2 * LANES>{});
            } else {
                prefetch_k(nxt, ic_all{}, ic_zero{});
            }
        }
        if (!TMA) cp_async_commit();        // group B (possibly empty): K~ of the next item
        // ---- inverse step 2: tasks (c, n2): R1-point over k1, rows n1 R2 + n2 (n1 < R1/2 when pruned) stored
#pragma unroll
        for (int it = 0; it < NT1; ++it) {
            const int task = tp + it * TPP;
            if ((3 * R2) % TPP == 0 || task < 3 * R2) {
                const int c = task / R2, n2 = task % R2;
                cx<T> w[R1];
                const cx<T>* src = buf + c * TILE + n2 * P1 * LANES + lane;
                static_for<R1>([&](auto pc) { w[decltype(pc)::value] = src[brev<R1>(decltype(pc)::value) * LANES]; });
                DitF<T, +1, R1, 0, false, PRUNE>::run(w);
                cx<T>* out = base + c * cs + (int64_t)n2 * sa;
                static_for<R1>([&](auto nc) {
                    constexpr int n1 = decltype(nc)::value;
                    if constexpr (!PRUNE || n1 < R1 / 2) {
                        if (!PRUNE || R2 * n1 + n2 < a.nz) out[(int64_t)(R2 * n1) * sa] = w[n1];
                    }
                });
            }
        }
        cur = nxt;
    }
    cp_async_wait<0>();
}

// Tensor maps of the tiled spectra S[b][c][g][z][ky][L] (as reals: 2 L per row) and of the tiled table Kt[6][g][ky][kz][L]
// with the boxes of one tile / one K~ tile.  False when the strides are not the tiled ones or the encoder is missing.
template <typename T>
static bool make_z_maps(void* S, const T* Kt, const Z2Args& a, int lanes, int nin, int hz, CUtensorMap* smap, CUtensorMap* kmap)
{
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn enc = nullptr;
    static bool tried = false;
    if (!tried) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) == cudaSuccess &&
            qr == cudaDriverEntryPointSuccess)
            enc = reinterpret_cast<encode_fn>(fn);
        tried = true;
    }
    if (!enc) return false;
    const int64_t L = lanes, My = a.My, nz = a.nz, G = a.ngroups, Hy = a.My / 2 + 1;
    if (a.s_ky != L || a.s_z != My * L || a.s_g != nz * My * L || a.cs != G * nz * My * L) return false;
    if (a.k_skz != L || a.k_sky != hz * L || a.k_sg != Hy * hz * L || a.kcs != G * Hy * hz * L) return false;
    if (hz > 256 || nin > 256) return false;
    const CUtensorMapDataType dt = sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    const cuuint32_t es[5] = {1, 1, 1, 1, 1};
    const cuuint64_t row = (cuuint64_t)(2 * L * sizeof(T));                               // 128 bytes
    const cuuint64_t sd[5] = {(cuuint64_t)(2 * L), (cuuint64_t)My, (cuuint64_t)nz, (cuuint64_t)G, (cuuint64_t)3 * a.batch};
    const cuuint64_t ss[4] = {row, row * My, row * My * nz, row * My * nz * G};
    const cuuint32_t sb[5] = {(cuuint32_t)(2 * L), 1, (cuuint32_t)nin, 1, 3};
    if (enc(smap, dt, 5, S, sd, ss, sb, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
            CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return false;
    const cuuint64_t krow = (cuuint64_t)(L * sizeof(T));
    const cuuint64_t kd[5] = {(cuuint64_t)L, (cuuint64_t)hz, (cuuint64_t)Hy, (cuuint64_t)G, 6};
    const cuuint64_t ks[4] = {krow, krow * hz, krow * hz * Hy, krow * hz * Hy * G};
    const cuuint32_t kb[5] = {(cuuint32_t)L, (cuuint32_t)hz, 1, 1, 6};
    return enc(kmap, dt, 5, const_cast<T*>(Kt), kd, ks, kb, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
               CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <typename T, int M, int LANES, bool PRUNE>
static cudaError_t launch_one(void* S, const T* Kt, Z2Args a, cudaStream_t st)
{
    using C = ZCfg<T, M, LANES, PRUNE>;
    static PerDevice<int> cache;
    int& nblocks = cache.here();
    if (!nblocks) {
        cudaError_t e = cudaFuncSetAttribute(k2_zmul<T, M, LANES, PRUNE, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)C::smem);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(k2_zmul<T, M, LANES, PRUNE, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem);
        if (e != cudaSuccess) return e;
        int dev = 0, sms = 0, per = 0;
        if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, k2_zmul<T, M, LANES, PRUNE, false>, C::THREADS, C::smem)) !=
            cudaSuccess)
            return e;
        nblocks = sms * (per > 0 ? per : 1);
    }
    a.nitems = a.ngroups * (a.My / 2 + 1);
    const int grid = a.nitems < nblocks ? a.nitems : nblocks;
    CUtensorMap smap, kmap;
    memset(&smap, 0, sizeof(smap));
    memset(&kmap, 0, sizeof(kmap));
    if (make_z_maps<T>(S, Kt, a, LANES, C::NIN, C::HZ, &smap, &kmap))
        k2_zmul<T, M, LANES, PRUNE, true><<<grid, C::THREADS, C::smem, st>>>(static_cast<cx<T>*>(S), Kt, a, smap, kmap);
    else
        k2_zmul<T, M, LANES, PRUNE, false><<<grid, C::THREADS, C::smem, st>>>(static_cast<cx<T>*>(S), Kt, a, smap, kmap);
    return cudaGetLastError();
}

template <typename T, int M, int LANES>
static cudaError_t launch_p(bool prune, void* S, const T* Kt, const Z2Args& a, cudaStream_t st)
{
    return prune ? launch_one<T, M, LANES, true>(S, Kt, a, st) : launch_one<T, M, LANES, false>(S, Kt, a, st);
}

}  // namespace v2

bool zmul2_supported(int M) { return M == 64 || M == 128 || M == 256; }

// fused z pass in place on the spectra; strides as in Z2Args (ngroups groups of 128 bytes of consecutive kx)
template <typename T>
cudaError_t launch_zmul2(const FftCtx& c, void* S, const T* Kt, const DevMember* members, int nz, int My, int ngroups,
                         int batch, const int64_t sstr[4], const int64_t kstr[4], const int perm[3], cudaStream_t st)
{
    const int M = c.plan[2].M;
    constexpr int L128 = 128 / (int)sizeof(v2::cx<T>);      // lanes of a 128-byte row
    // slot order of ky: radices of the three-level y pass (powers of two), or natural order
    int lg[3] = {-1, 0, 0};
    if (perm[0]) {
        for (int i = 0; i < 3; ++i) {
            if (perm[i] <= 0 || (perm[i] & (perm[i] - 1))) return cudaErrorInvalidValue;
            lg[i] = 0;
            while ((1 << lg[i]) < perm[i]) ++lg[i];
        }
    }
    v2::Z2Args a{c.tw, members, My, batch, nz, ngroups, 0, sstr[0], sstr[1], sstr[2], sstr[3],
                 kstr[0], kstr[1], kstr[2], kstr[3], lg[0], lg[1], lg[2]};
    const bool prune = 2 * nz <= M;              // zero-padded axis
    if (!prune && nz != M) return cudaErrorInvalidValue;
    switch (M) {
        case 64: return v2::launch_p<T, 64, L128>(prune, S, Kt, a, st);
        case 128: return v2::launch_p<T, 128, L128>(prune, S, Kt, a, st);
        // 128-byte rows (one 256-thread block per SM) beat 64-byte rows (two 128-thread blocks): 0.66 vs 0.80 ms at cfg5a
        case 256: return v2::launch_p<T, 256, L128>(prune, S, Kt, a, st);
        default: return cudaErrorInvalidValue;
    }
}

template cudaError_t launch_zmul2<double>(const FftCtx&, void*, const double*, const DevMember*, int, int, int, int,
                                          const int64_t*, const int64_t*, const int*, cudaStream_t);
template cudaError_t launch_zmul2<float>(const FftCtx&, void*, const float*, const DevMember*, int, int, int, int,
                                         const int64_t*, const int64_t*, const int*, cudaStream_t);

}  // namespace fe
