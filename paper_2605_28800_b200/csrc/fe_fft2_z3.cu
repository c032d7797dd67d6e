// fe_fft2_z3.cu -- fused z pass on MIRROR PAIRS of tiles (Eq. 5-6 in k-space) for
// the zero-padded z axis of transform length 256 (config 5a): forward z transform, E~_i = -escale sum_j K~_ij P~_j,
// inverse z transform, in place on the spectra, like k2_zmul (fe_fft2_z.cu) but organised so that every warp has the
// same amount of work in every phase and shared-memory and fp64 phases of different warps overlap:
//
//   unit      = the tiles ky and My - ky of one (kx group, batch member): they share the K~ values (up to the signs of
//               the odd components), which a thread loads ONCE into registers for both;
//   columns   = (tile, component, n2): 48 per kx lane.  The 256-point transform is 32 x 8: a column's 32-point step is
//               done by one thread in registers, the 8-point step + multiply + inverse 8-point step by the thread of k1;
//   exchange  = ONE buffer [tile][c][k1 * 8 + n2][lane] used in place by all steps: the thread of k1 reads and writes
//               exactly its own rows, a column task reads (inverse) or writes (forward) exactly its own column;
//   E phase   = inverse 32-point step of the unit just multiplied (column -> global rows) followed by the forward
//               32-point step of the NEXT unit (global rows -> the same column): 48 column groups of work items on NW
//               warps = three per warp, no staging buffer;  M phase = two k1 work items (one per tile) per thread.
// Two block barriers per unit (E | M); inside the E phase warps run three tasks each without meeting, in different
// orders on the two warps of a scheduler, so loads, stores and arithmetic of different warps interleave.
#include "fe_fft2.cuh"

namespace fe {
namespace v2 {

struct Z3Args {
    const void* tw;
    const DevMember* members;
    int My, batch, nz, ngroups, nunits;
    int64_t cs, s_z, s_ky, s_g;          // spectrum strides (complex elements), see Z2Args in fe_fft2_z.cu
    int64_t kcs, k_skz, k_sky, k_sg;     // tensor strides (real elements)
    int la, lb, lc;                      // slot order of ky (binary logarithms of the radices), la < 0: natural
};

template <typename T> struct Z3Cfg {
    static constexpr int M = 256, R1 = 32, R2 = 8;
    static constexpr int LANES = 128 / (int)sizeof(cx<T>);
    static constexpr int THREADS = LANES * R1;
    static constexpr int NW = THREADS / 32, HALF = NW / 2;
    static constexpr int TPW = 32 / LANES;                 // columns of a warp task
    static constexpr int CQT = 3 * R2 / TPW;               // column groups per tile
    static constexpr int TILE = 3 * M * LANES;             // complex elements of one tile in the exchange buffer
    static constexpr size_t smem = (size_t)2 * TILE * sizeof(cx<T>);
    static_assert(2 * CQT == NW + HALF, "48 columns x LANES = three column-group tasks per warp and direction pair");
};

__device__ __forceinline__ double z3_xorsign(double x, unsigned s)
{
    return __hiloint2double(__double2hiint(x) ^ (int)s, __double2loint(x));
}
__device__ __forceinline__ float z3_xorsign(float x, unsigned s) { return __uint_as_float(__float_as_uint(x) ^ s); }
__device__ __forceinline__ void z3_arrive(int id) { asm volatile("bar.arrive %0, 64;\n" ::"r"(id) : "memory"); }
__device__ __forceinline__ void z3_sync(int id) { asm volatile("bar.sync %0, 64;\n" ::"r"(id) : "memory"); }
// per-thread prefetch of the line at p into L2 (the bulk form runs on the uniform datapath: a warp whose lanes hold
// different addresses serialises over its lanes)
__device__ __forceinline__ void z3_prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];\n" ::"l"(p)); }

template <typename T> struct Z3Unit {
    cx<T>* base0;         // first element of tile ky (kx lane 0, component 0, row 0)
    cx<T>* base1;         // ... of tile My - ky
    const T* kbase;       // K~ of the item (kz = 0, component 0, kx lane 0)
    int b;
    bool hasB, valid;
};

// FULLZ: the axis carries exactly M / 2 data rows (no row predicate anywhere)
template <typename T, bool FULLZ>
__global__ void __launch_bounds__(Z3Cfg<T>::THREADS, 1) k3_zmul(cx<T>* S, const T* __restrict__ Kt, Z3Args a)
{
    using C = Z3Cfg<T>;
    constexpr int M = C::M, R1 = C::R1, R2 = C::R2, LANES = C::LANES, NW = C::NW, HALF = C::HALF, TPW = C::TPW;
    constexpr int CQT = C::CQT, TILE = C::TILE;
    cx<T>* buf = reinterpret_cast<cx<T>*>(fe2_smem);
    const int lane = threadIdx.x % LANES, tp = threadIdx.x / LANES, warp = threadIdx.x / 32, sub = tp % TPW;
    const int64_t cs = a.cs, sz = a.s_z;

    auto decode = [&](int u) {
        Z3Unit<T> un;
        un.valid = u >= 0 && u < a.nunits;
        un.hasB = false;
        un.b = 0;
        un.base0 = un.base1 = S;
        un.kbase = Kt;
        if (!un.valid) return un;
        const int item = u / a.batch;
        un.b = u - item * a.batch;
        const int kyh = item / a.ngroups, kxg = item - kyh * a.ngroups;
        un.hasB = kyh != 0 && 2 * kyh != a.My;
        auto slot = [&](int ky) {
            if (a.la < 0) return ky;
            return ((ky & ((1 << a.la) - 1)) << (a.lb + a.lc)) | (((ky >> a.la) & ((1 << a.lb) - 1)) << a.lc) |
                   (ky >> (a.la + a.lb));
        };
        cx<T>* s0 = S + (int64_t)un.b * 3 * cs + (int64_t)kxg * a.s_g;
        un.base0 = s0 + (int64_t)slot(kyh) * a.s_ky;
        un.base1 = s0 + (int64_t)slot(un.hasB ? a.My - kyh : kyh) * a.s_ky;
        un.kbase = Kt + (int64_t)kyh * a.k_sky + (int64_t)kxg * a.k_sg;
        return un;
    };
    // inverse 32-point step of column group q: exchange column -> rows n2 + 8 n1 (n1 < 16) of the tile in memory
    auto taskU = [&](const Z3Unit<T>& un, int q) {
        const int tile = q / CQT;
        if (!un.valid || (tile && !un.hasB)) return;
        const int col = (q - tile * CQT) * TPW + sub, c = col >> 3, n2 = col & 7;
        const cx<T>* src = buf + tile * TILE + (c * M + n2) * LANES + lane;
        cx<T> w[R1];
        static_for<R1>([&](auto pc) { w[decltype(pc)::value] = src[brev<R1>(decltype(pc)::value) * R2 * LANES]; });
        DitF<T, +1, R1, 0, false, true>::run(w);
        cx<T>* out = (tile ? un.base1 : un.base0) + lane + c * cs + (int64_t)n2 * sz;
        static_for<R1 / 2>([&](auto nc) {
            constexpr int n1 = decltype(nc)::value;
            if (FULLZ || R2 * n1 + n2 < a.nz) out[(int64_t)(R2 * n1) * sz] = w[n1];
        });
    };
    // forward 32-point step of column group q: rows of the tile in memory -> exchange column
    auto taskT = [&](const Z3Unit<T>& un, int q) {
        const int tile = q / CQT;
        if (!un.valid || (tile && !un.hasB)) return;
        const int col = (q - tile * CQT) * TPW + sub, c = col >> 3, n2 = col & 7;
        const cx<T>* in = (tile ? un.base1 : un.base0) + lane + c * cs + (int64_t)n2 * sz;
        cx<T> w[R1];
        static_for<R1>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            constexpr int n1 = brev<R1>(p);
            if constexpr (n1 < R1 / 2) {
                if constexpr (FULLZ) {
                    w[p] = in[(int64_t)(R2 * n1) * sz];
                } else {
                    const bool ok = R2 * n1 + n2 < a.nz;      // rows beyond nz are read at row n2 and replaced by zero
                    const cx<T> v = in[ok ? (int64_t)(R2 * n1) * sz : 0];
                    w[p] = {ok ? v.x : (T)0, ok ? v.y : (T)0};
                }
            }
        });
        DitF<T, -1, R1, 0, true, false>::run(w);
        cx<T>* dst = buf + tile * TILE + (c * M + n2) * LANES + lane;
        static_for<R1>([&](auto kc) { dst[decltype(kc)::value * R2 * LANES] = w[decltype(kc)::value]; });
    };

    const int k1 = tp;
    auto phaseM = [&](const Z3Unit<T>& un) {
        // K~ of the thread's eight frequencies kz = k1 + 32 k2, loaded once for both tiles of the unit
        T Kv[R2][6];
        static_for<R2>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            constexpr int k2 = brev<R2>(p);
            const int kz = k1 + R1 * k2;
            const int kzm = 2 * kz <= M ? kz : M - kz;
            const T* kp = un.kbase + (int64_t)kzm * a.k_skz + lane;
#pragma unroll
            for (int c6 = 0; c6 < 6; ++c6) Kv[p][c6] = kp[c6 * a.kcs];
        });
        const T esc = (T)(-a.members[un.b].escale);
        // inter-step twiddles of the thread of k1: w_M^(n2 k1) (seven L1-resident loads per unit; keeping them in
        // registers across the E phase would push its 32-point tasks into spills)
        cx<T> wk[R2];
        {
            const cx<T>* twg = static_cast<const cx<T>*>(a.tw);
            static_for<R2 - 1>([&](auto nc) {
                constexpr int n2 = decltype(nc)::value + 1;
                wk[n2] = twg[(n2 * k1) * (kTwiddleN / M)];
            });
        }
#pragma unroll 1
        for (int tile = 0; tile < 2; ++tile) {
            if (tile && !un.hasB) break;
            const unsigned sy = tile ? 0x80000000u : 0u;      // tile 1 is ky > My / 2: xy and yz change sign
            cx<T>* row = buf + tile * TILE + (k1 * R2) * LANES + lane;
            cx<T> u[3][R2];
#pragma unroll
            for (int c = 0; c < 3; ++c)
                static_for<R2>([&](auto nc) { u[c][decltype(nc)::value] = row[(c * M + decltype(nc)::value) * LANES]; });
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                static_for<R2 - 1>([&](auto nc) {
                    constexpr int n2 = decltype(nc)::value + 1;
                    u[c][n2] = cmul(u[c][n2], wk[n2]);
                });
                Dif<T, -1, R2>::run(u[c]);
            }
            if (tile == 0) {
                // first use of K~ (it has arrived behind the forward step): -1/(eps0 epsB) of Eq. 6 rides on it, and
                // the components that are odd in kz (xz, yz) take their sign
                static_for<R2>([&](auto pc) {
                    constexpr int p = decltype(pc)::value;
                    constexpr int k2 = brev<R2>(p);
                    const unsigned sgn = 2 * (k1 + R1 * k2) > M ? 0x80000000u : 0u;
#pragma unroll
                    for (int c6 = 0; c6 < 6; ++c6) Kv[p][c6] *= esc;
                    Kv[p][4] = z3_xorsign(Kv[p][4], sgn);
                    Kv[p][5] = z3_xorsign(Kv[p][5], sgn);
                });
            }
            static_for<R2>([&](auto pc) {
                constexpr int p = decltype(pc)::value;
                const T Kxx = Kv[p][0], Kyy = Kv[p][1], Kzz = Kv[p][2];
                const T Kxy = z3_xorsign(Kv[p][3], sy), Kxz = Kv[p][4], Kyz = z3_xorsign(Kv[p][5], sy);
                const cx<T> Px = u[0][p], Py = u[1][p], Pz = u[2][p];
                u[0][p] = {Kxx * Px.x + Kxy * Py.x + Kxz * Pz.x, Kxx * Px.y + Kxy * Py.y + Kxz * Pz.y};
                u[1][p] = {Kxy * Px.x + Kyy * Py.x + Kyz * Pz.x, Kxy * Px.y + Kyy * Py.y + Kyz * Pz.y};
                u[2][p] = {Kxz * Px.x + Kyz * Py.x + Kzz * Pz.x, Kxz * Px.y + Kyz * Py.y + Kzz * Pz.y};
            });
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                DitF<T, +1, R2>::run(u[c]);
                static_for<R2>([&](auto nc) {
                    constexpr int n2 = decltype(nc)::value;
                    cx<T> val = u[c][n2];
                    if constexpr (n2 != 0) val = cmulc(val, wk[n2]);
                    row[(c * M + n2) * LANES] = val;
                });
            }
        }
    };
    // rows of a unit two steps ahead -> L2 (the forward column tasks read them straight from global memory)
    auto prefetch_rows = [&](const Z3Unit<T>& un) {
        if (!un.valid) return;
        constexpr int per_tile = 3 * (M / 2);
        for (int r = threadIdx.x; r < 2 * per_tile; r += C::THREADS) {
            const int tile = r / per_tile, rr = r - tile * per_tile, c = rr / (M / 2), z = rr - c * (M / 2);
            if ((tile && !un.hasB) || (!FULLZ && z >= a.nz)) continue;
            z3_prefetch_l2((tile ? un.base1 : un.base0) + c * cs + (int64_t)z * sz);
        }
        // K~ rows of the unit's item: 6 components x (M/2 + 1) rows of LANES reals
        for (int r = threadIdx.x; r < 6 * (M / 2 + 1); r += C::THREADS) {
            const int c6 = r / (M / 2 + 1), kz = r - c6 * (M / 2 + 1);
            z3_prefetch_l2(un.kbase + c6 * a.kcs + (int64_t)kz * a.k_skz);
        }
    };

    int u0 = blockIdx.x;
    Z3Unit<T> prev = decode(-1), next = decode(u0);
    prefetch_rows(decode(u0 + (int)gridDim.x));
    while (prev.valid || next.valid) {
        // ---- E phase: inverse step of `prev`, forward step of `next`; column group s of both belongs to one warp,
        // except the groups NW .. NW + HALF - 1 whose inverse step is done by warp s - NW and whose forward step by
        // warp s - NW + HALF (ordered by a two-warp barrier)
        if (warp < HALF) {
            taskU(prev, NW + warp);
            z3_arrive(1 + warp);
            taskU(prev, warp);
            taskT(next, warp);
        } else {
            taskU(prev, warp);
            taskT(next, warp);
            z3_sync(1 + warp - HALF);
            taskT(next, NW + warp - HALF);
        }
        __syncthreads();
        if (!next.valid) break;
        u0 += gridDim.x;
        prefetch_rows(decode(u0 + (int)gridDim.x));
        phaseM(next);
        prev = next;
        next = decode(u0);
        __syncthreads();
    }
}


// ------------------------------------------------------------------------------------------------------------------
// k5_zmul: ONE tile at a time with the in-place column layout above, cp.async staging of the next tile's rows and the
// K~ tile of the item in shared memory (as k2_zmul).  Per tile two phases and two block barriers:
//   M phase  8-point step + multiply + inverse 8-point step of the current tile, every thread its k1, in place;
//   E phase  inverse 32-point step of the current tile (column -> global rows) and forward 32-point step of the NEXT
//            tile (staged rows -> the same column): 2 CQT warp tasks on NW warps.  Warp w < NW/2 does both steps of
//            column group w; the remaining NW/4 groups have their inverse step done by warps NW/2 .. and their forward
//            step by the last NW/4 warps (ordered by a two-warp barrier): every scheduler gets three 32-point tasks,
//            where the three-phase kernel gives two of the four schedulers four.
// ------------------------------------------------------------------------------------------------------------------
template <typename T> struct Z5Cfg {
    static constexpr int M = 256, R1 = 32, R2 = 8, HZ = M / 2 + 1, NIN = M / 2;
    static constexpr int LANES = 128 / (int)sizeof(cx<T>);
    static constexpr int THREADS = LANES * R1;
    static constexpr int NW = THREADS / 32, HALF = NW / 2, Q = NW / 4;
    static constexpr int TPW = 32 / LANES;
    static constexpr int CQT = 3 * R2 / TPW;
    static constexpr int TILE = 3 * M * LANES;
    static constexpr size_t ex_bytes = (size_t)TILE * sizeof(cx<T>);
    static constexpr size_t st_bytes = (size_t)3 * NIN * LANES * sizeof(cx<T>);
    static constexpr size_t k_bytes = ((size_t)6 * HZ * LANES * sizeof(T) + 15) / 16 * 16;
    static constexpr size_t tw_bytes = (size_t)(R2 - 1) * R1 * sizeof(cx<T>);       // w_M^(n2 k1) at [n2 - 1][k1]
    static constexpr size_t smem = ex_bytes + st_bytes + k_bytes + tw_bytes;
    static_assert(CQT == HALF + Q, "24 columns x LANES = HALF + Q column groups");
};

__device__ __forceinline__ void z5_cp16(void* smem, const void* gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void z5_commit() { asm volatile("cp.async.commit_group;\n" ::); }
__device__ __forceinline__ void z5_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }

struct Z5It {
    int item, b, m;
};

template <typename T, bool FULLZ>
__global__ void __launch_bounds__(Z5Cfg<T>::THREADS, 1) k5_zmul(cx<T>* S, const T* __restrict__ Kt, Z3Args a)
{
    using C = Z5Cfg<T>;
    constexpr int M = C::M, R1 = C::R1, R2 = C::R2, LANES = C::LANES, NW = C::NW, HALF = C::HALF, Q = C::Q, TPW = C::TPW;
    constexpr int HZ = C::HZ, NIN = C::NIN;
    cx<T>* buf = reinterpret_cast<cx<T>*>(fe2_smem);                       // exchange [3][k1 * 8 + n2][LANES]
    cx<T>* stage = buf + C::TILE;                                          // staged rows [3][NIN][LANES]
    T* kbuf = reinterpret_cast<T*>(stage + 3 * NIN * LANES);               // K~ tile [6][HZ][LANES]
    cx<T>* twk = reinterpret_cast<cx<T>*>(reinterpret_cast<unsigned char*>(kbuf) + C::k_bytes);   // [R2 - 1][R1]
    const int lane = threadIdx.x % LANES, tp = threadIdx.x / LANES, warp = threadIdx.x / 32, sub = tp % TPW;
    const int64_t cs = a.cs, sz = a.s_z;
    const int nitems = a.ngroups * (a.My / 2 + 1);

    auto valid = [&](const Z5It& it) { return it.item < nitems; };
    auto mirrors = [&](int item) {
        const int kyh = item / a.ngroups;
        return (kyh == 0 || 2 * kyh == a.My) ? 1 : 2;
    };
    auto advance = [&](Z5It it) {
        if (++it.m < mirrors(it.item)) return it;
        it.m = 0;
        if (++it.b < a.batch) return it;
        it.b = 0;
        it.item += gridDim.x;
        return it;
    };
    auto tile_base = [&](const Z5It& it) -> cx<T>* {
        const int kyh = it.item / a.ngroups, kxg = it.item - kyh * a.ngroups;
        const int ky = it.m ? a.My - kyh : kyh;
        int slot = ky;
        if (a.la >= 0)
            slot = ((ky & ((1 << a.la) - 1)) << (a.lb + a.lc)) | (((ky >> a.la) & ((1 << a.lb) - 1)) << a.lc) |
                   (ky >> (a.la + a.lb));
        return S + (int64_t)it.b * 3 * cs + (int64_t)slot * a.s_ky + (int64_t)kxg * a.s_g;
    };
    // asynchronous copies: data rows of a tile -> stage, K~ tile of an item -> kbuf (16 bytes per copy)
    auto prefetch_tile = [&](const cx<T>* tb) {
        constexpr int PER = 16 / (int)sizeof(cx<T>), OPS_ROW = LANES / PER, RSTEP = C::THREADS / OPS_ROW;
        static_assert(NIN % RSTEP == 0, "tile copy must be regular");
        const int q = threadIdx.x % OPS_ROW, row0 = threadIdx.x / OPS_ROW;
        const cx<T>* g = tb + (int64_t)row0 * sz + q * PER;
        cx<T>* s = stage + row0 * LANES + q * PER;
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int j = 0; j < NIN / RSTEP; ++j)
                if (FULLZ || row0 + j * RSTEP < a.nz)
                    z5_cp16(s + (c * NIN + j * RSTEP) * LANES, g + c * cs + (int64_t)(j * RSTEP) * sz);
    };
    auto prefetch_k = [&](int item) {
        constexpr int PER = 16 / (int)sizeof(T), OPS_ROW = LANES / PER, RSTEP = C::THREADS / OPS_ROW;
        const int kyh = item / a.ngroups, kxg = item - kyh * a.ngroups;
        const int q = threadIdx.x % OPS_ROW, row0 = threadIdx.x / OPS_ROW;
        const T* g = Kt + (int64_t)kyh * a.k_sky + (int64_t)kxg * a.k_sg + (int64_t)row0 * a.k_skz + q * PER;
        T* s = kbuf + row0 * LANES + q * PER;
#pragma unroll
        for (int c6 = 0; c6 < 6; ++c6)
#pragma unroll
            for (int j = 0; j < (HZ + RSTEP - 1) / RSTEP; ++j)
                if (row0 + j * RSTEP < HZ)
                    z5_cp16(s + (c6 * HZ + j * RSTEP) * LANES, g + c6 * a.kcs + (int64_t)(j * RSTEP) * a.k_skz);
    };
    // inverse 32-point step of column group q of the current tile: exchange column -> rows of the tile in memory
    auto taskU = [&](cx<T>* tb, int q) {
        const int col = q * TPW + sub, c = col >> 3, n2 = col & 7;
        const cx<T>* src = buf + (c * M + n2) * LANES + lane;
        cx<T> w[R1];
        static_for<R1>([&](auto pc) { w[decltype(pc)::value] = src[brev<R1>(decltype(pc)::value) * R2 * LANES]; });
        DitF<T, +1, R1, 0, false, true>::run(w);
        cx<T>* out = tb + lane + c * cs + (int64_t)n2 * sz;
        static_for<R1 / 2>([&](auto nc) {
            constexpr int n1 = decltype(nc)::value;
            if (FULLZ || R2 * n1 + n2 < a.nz) out[(int64_t)(R2 * n1) * sz] = w[n1];
        });
    };
    // forward 32-point step of column group q of the next tile: staged rows -> exchange column
    auto taskT = [&](int q) {
        const int col = q * TPW + sub, c = col >> 3, n2 = col & 7;
        const cx<T>* src = stage + (c * NIN + n2) * LANES + lane;
        cx<T> w[R1];
        static_for<R1>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            constexpr int n1 = brev<R1>(p);
            if constexpr (n1 < R1 / 2) w[p] = src[n1 * R2 * LANES];
        });
        DitF<T, -1, R1, 0, true, false>::run(w);
        cx<T>* dst = buf + (c * M + n2) * LANES + lane;
        static_for<R1>([&](auto kc) { dst[decltype(kc)::value * R2 * LANES] = w[decltype(kc)::value]; });
    };
    const int k1 = tp;
    auto phaseM = [&](const Z5It& it, const T esc) {
        cx<T> wk[R2];
        static_for<R2 - 1>([&](auto nc) { wk[decltype(nc)::value + 1] = twk[decltype(nc)::value * R1 + k1]; });
        const unsigned sy = it.m ? 0x80000000u : 0u;          // mirror tile: ky > My / 2, xy and yz change sign
        cx<T>* row = buf + (k1 * R2) * LANES + lane;
        cx<T> u[3][R2];
#pragma unroll
        for (int c = 0; c < 3; ++c)
            static_for<R2>([&](auto nc) { u[c][decltype(nc)::value] = row[(c * M + decltype(nc)::value) * LANES]; });
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            static_for<R2 - 1>([&](auto nc) {
                constexpr int n2 = decltype(nc)::value + 1;
                u[c][n2] = cmul(u[c][n2], wk[n2]);
            });
            Dif<T, -1, R2>::run(u[c]);
        }
        static_for<R2>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            constexpr int k2 = brev<R2>(p);
            const int kz = k1 + R1 * k2;
            const int kzm = 2 * kz <= M ? kz : M - kz;
            const unsigned sgn = 2 * kz > M ? 0x80000000u : 0u;
            const T* kp = kbuf + kzm * LANES + lane;
            const T Kxx = kp[0], Kyy = kp[HZ * LANES], Kzz = kp[2 * HZ * LANES];
            const T Kxy = z3_xorsign(kp[3 * HZ * LANES], sy), Kxz = z3_xorsign(kp[4 * HZ * LANES], sgn);
            const T Kyz = z3_xorsign(kp[5 * HZ * LANES], sy ^ sgn);
            const cx<T> Px = u[0][p], Py = u[1][p], Pz = u[2][p];
            u[0][p] = {Kxx * Px.x + Kxy * Py.x + Kxz * Pz.x, Kxx * Px.y + Kxy * Py.y + Kxz * Pz.y};
            u[1][p] = {Kxy * Px.x + Kyy * Py.x + Kyz * Pz.x, Kxy * Px.y + Kyy * Py.y + Kyz * Pz.y};
            u[2][p] = {Kxz * Px.x + Kyz * Py.x + Kzz * Pz.x, Kxz * Px.y + Kyz * Py.y + Kzz * Pz.y};
        });
        // -1/(eps0 epsB) of Eq. 6 rides on the inverse twiddles
        static_for<R2 - 1>([&](auto nc) {
            constexpr int n2 = decltype(nc)::value + 1;
            wk[n2] = {esc * wk[n2].x, esc * wk[n2].y};
        });
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            DitF<T, +1, R2>::run(u[c]);
            static_for<R2>([&](auto nc) {
                constexpr int n2 = decltype(nc)::value;
                cx<T> val = u[c][n2];
                if constexpr (n2 != 0) val = cmulc(val, wk[n2]);
                else val = {esc * val.x, esc * val.y};
                row[(c * M + n2) * LANES] = val;
            });
        }
    };

    Z5It cur{(int)blockIdx.x, 0, 0};
    if (!valid(cur)) return;
    if (!FULLZ) {                           // rows nz .. M/2 of the staged half: cleared once, never written again
        for (int e = threadIdx.x; e < 3 * NIN * LANES; e += C::THREADS) stage[e] = cx<T>{0, 0};
        __syncthreads();
    }
    for (int e = threadIdx.x; e < (R2 - 1) * R1; e += C::THREADS)
        twk[e] = static_cast<const cx<T>*>(a.tw)[((e / R1 + 1) * (e % R1)) * (kTwiddleN / M)];
    cx<T>* cur_base = tile_base(cur);
    T esc_cur = (T)(-a.members[cur.b].escale), esc_nxt = esc_cur;
    prefetch_tile(cur_base);
    prefetch_k(cur.item);
    z5_commit();
    z5_wait_all();
    __syncthreads();
    // prologue E phase: forward step of the first tile only
    if (warp < HALF) taskT(warp);
    else if (warp >= HALF + Q) taskT(warp - Q);
    Z5It nxt = advance(cur);
    cx<T>* nxt_base = valid(nxt) ? tile_base(nxt) : cur_base;
    if (valid(nxt)) esc_nxt = (T)(-a.members[nxt.b].escale);
    __syncthreads();
    if (valid(nxt)) prefetch_tile(nxt_base);
    z5_commit();
    while (true) {
        phaseM(cur, esc_cur);
        z5_wait_all();                      // rows of the next tile have landed ...
        __syncthreads();                    // ... for every thread; exchange holds the inverse-ready tile; K~ tile free
        const bool more = valid(nxt);
        if (more && nxt.item != cur.item) prefetch_k(nxt.item);
        z5_commit();
        if (warp < HALF) {
            taskU(cur_base, warp);
            if (more) taskT(warp);
        } else if (warp < HALF + Q) {
            taskU(cur_base, warp);
            z3_arrive(1 + warp - HALF);
        } else {
            z3_sync(1 + warp - HALF - Q);
            if (more) taskT(warp - Q);
        }
        if (!more) break;
        cur = nxt;
        cur_base = nxt_base;
        esc_cur = esc_nxt;
        nxt = advance(cur);
        if (valid(nxt)) {
            nxt_base = tile_base(nxt);
            esc_nxt = (T)(-a.members[nxt.b].escale);
        }
        z5_wait_all();                      // K~ of the tile about to be multiplied
        __syncthreads();                    // exchange holds the forward-ready tile; staging buffer free
        if (valid(nxt)) prefetch_tile(nxt_base);
        z5_commit();
    }
}

}  // namespace v2

// paired fused z pass; same argument meaning as launch_zmul2 (fe_fft2_z.cu).  Only the zero-padded 256-point axis.
bool zmul3_supported(int M, int nz) { return M == 256 && 2 * nz <= M; }

template <typename T>
cudaError_t launch_zmul3(const FftCtx& c, void* S, const T* Kt, const DevMember* members, int nz, int My, int ngroups,
                         int batch, const int64_t sstr[4], const int64_t kstr[4], const int perm[3], int variant,
                         cudaStream_t st)
{
    using C = v2::Z3Cfg<T>;
    if (!zmul3_supported(c.plan[2].M, nz)) return cudaErrorInvalidValue;
    int lg[3] = {-1, 0, 0};
    if (perm[0]) {
        for (int i = 0; i < 3; ++i) {
            if (perm[i] <= 0 || (perm[i] & (perm[i] - 1))) return cudaErrorInvalidValue;
            lg[i] = 0;
            while ((1 << lg[i]) < perm[i]) ++lg[i];
        }
    }
    static PerDevice<int> cache;
    int& nblocks = cache.here();
    if (!nblocks) {
        cudaError_t e = cudaFuncSetAttribute(v2::k3_zmul<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(v2::k3_zmul<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem);
        if (e != cudaSuccess) return e;
        int dev = 0, sms = 0;
        if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        nblocks = sms;
    }
    const int nunits = ngroups * (My / 2 + 1) * batch;
    v2::Z3Args a{c.tw, members, My, batch, nz, ngroups, nunits, sstr[0], sstr[1], sstr[2], sstr[3],
                 kstr[0], kstr[1], kstr[2], kstr[3], lg[0], lg[1], lg[2]};
    const int grid = nunits < nblocks ? nunits : nblocks;
    if (variant == 2) {
        using C5 = v2::Z5Cfg<T>;
        static PerDevice<int> cache5;
        int& conf = cache5.here();
        if (!conf) {
            cudaError_t e = cudaFuncSetAttribute(v2::k5_zmul<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C5::smem);
            if (e == cudaSuccess)
                e = cudaFuncSetAttribute(v2::k5_zmul<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C5::smem);
            if (e != cudaSuccess) return e;
            conf = 1;
        }
        const int nitems = ngroups * (My / 2 + 1);
        const int grid5 = nitems < nblocks ? nitems : nblocks;
        if (2 * nz == C5::M) v2::k5_zmul<T, true><<<grid5, C5::THREADS, C5::smem, st>>>(static_cast<v2::cx<T>*>(S), Kt, a);
        else v2::k5_zmul<T, false><<<grid5, C5::THREADS, C5::smem, st>>>(static_cast<v2::cx<T>*>(S), Kt, a);
        return cudaGetLastError();
    }
    if (2 * nz == C::M) v2::k3_zmul<T, true><<<grid, C::THREADS, C::smem, st>>>(static_cast<v2::cx<T>*>(S), Kt, a);
    else v2::k3_zmul<T, false><<<grid, C::THREADS, C::smem, st>>>(static_cast<v2::cx<T>*>(S), Kt, a);
    return cudaGetLastError();
}

template cudaError_t launch_zmul3<double>(const FftCtx&, void*, const double*, const DevMember*, int, int, int, int,
                                          const int64_t*, const int64_t*, const int*, int, cudaStream_t);
template cudaError_t launch_zmul3<float>(const FftCtx&, void*, const float*, const DevMember*, int, int, int, int,
                                         const int64_t*, const int64_t*, const int*, int, cudaStream_t);

}  // namespace fe
