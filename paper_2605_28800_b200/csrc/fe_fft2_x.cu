// fe_fft2_x.cu -- size-specialised x passes: real rows of n_x
// values (zero-padded to m_x = 2 M when the axis is open) <-> half spectra X[0..M].
// The real transform of length 2 M runs as a complex transform of length M on z[j] = x[2j] + i x[2j+1]:
//   forward  Z = FFT_M(z);  X[k] = (Z[k] + conj Z[M-k])/2 - (i/2) w_2M^k (Z[k] - conj Z[M-k])
//   inverse  Z[k] = (X[k] + conj X[M-k])/2 + (i/2) conj(w_2M^k) (X[k] - conj X[M-k]);  z = M * IFFT_M(Z)
// (the inverse is unnormalised; 1/(M m_y m_z) is folded into the tensor spectrum at precompute).
// Each row is handled by R2 threads with the register two-level transform of fe_fft2.cuh.
#include "fe_fft2.cuh"
#include <string.h>
#include <cuda.h>          // CUtensorMap and cuTensorMapEncodeTiled's signature only; the entry point is fetched at run time

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
    // k6_xinv on a slab of z planes: plane q of the launch reads spectrum plane (q / pl_n) * pl_full + pl_off + q % pl_n
    // (pl_n planes of each of the B * 3 components, starting at z = pl_off of pl_full) and writes real plane
    // (q / pl_n) * pl_full + q % pl_n (the first pl_n planes of the component's region); pl_n == 0: q itself for both
    int pl_n, pl_full, pl_off;
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

// ------------------------------------------------------------------------------------------------------------------
// k6_xinv: persistent inverse x pass for the tiled spectrum layout (Mc = R2 * R2: 256 in fp64 / fp32, 64 in fp64), no block
// barrier in its loop.  A warp owns 32 / R2 rows of a group of ROWS rows (two at Mc = 256, described here): their half spectra ([g][row][L] in memory: a 3-D box of 2 rows) arrive by one
// tensor copy on the warp's own mbarrier into the warp's own buffer and are transformed IN PLACE there: a row's R2 threads
// own the row's 128-byte pieces, so the exchange of the two-level transform needs only __syncwarp, and an XOR swizzle
// (column ^ (row of the exchange & 7)) replaces the padding column, which lets the 16 x 16 exchange fit into the 33 x 8
// slots of the row.  As soon as every thread of the warp holds its second-step inputs the buffer is free and lane 0
// starts the copy of the warp's rows of the block's next group, which lands behind the second register FFT and the stores.
// ------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned x6_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

template <typename T, int M, bool PRUNE>
__global__ void __launch_bounds__(256, 2) k6_xinv(T* __restrict__ out, X2Args a, int G, int nplanes,
                                                  const __grid_constant__ CUtensorMap imap)
{
    using C = XCfg<M>;
    constexpr int R1 = C::R1, R2 = C::R2, TPP = C::TPP, ROWS = C::ROWS, TWG = 8;
    constexpr int L = 128 / (int)sizeof(cx<T>);                           // complex per 128-byte piece
    constexpr int SW = R2 < L ? R2 : L;                                   // the swizzle permutes within pieces
    constexpr int NT3 = R1 / TPP;                                         // second-step tasks (exchange rows tp + it TPP) per thread
    static_assert(R1 % TPP == 0 && R2 % L == 0 && (NT3 == 1 || TPP % 8 == 0), "an exchange row is whole pieces");
    constexpr int WR = 32 / TPP;                                          // rows per warp
    cx<T>* buf = reinterpret_cast<cx<T>*>(fe2_smem);                       // [warp][G][WR][L]
    cx<T>* tw = buf + (size_t)G * ROWS * L;                               // w_M^(n2 k1) at [k1 * R2 + n2]
    cx<T>* tws = tw + M;                                                  // w_2M^k
    const int t = threadIdx.x, tp = t % TPP, rl = t / TPP, warp = t >> 5;
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(tws + M) + warp;     // the warp's mbarrier
    cx<T>* wbuf = buf + (size_t)warp * G * WR * L;
    const int gpp = a.ny / ROWS;                                          // row groups per plane
    const int ngroups = nplanes * gpp;
    const unsigned bytes = (unsigned)((size_t)G * WR * L * sizeof(cx<T>));
    auto issue = [&](int grp) {
        int plane = grp / gpp;
        const int y0 = (grp - plane * gpp) * ROWS;
        if (a.pl_n) plane = (plane / a.pl_n) * a.pl_full + a.pl_off + plane % a.pl_n;
        // the warp's generic-proxy reads and exchange writes of the buffer are ordered before the copy engine's writes
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(x6_smem_u32(bar)), "r"(bytes) : "memory");
        asm volatile(
            "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];\n" ::"r"(
                x6_smem_u32(wbuf)),
            "l"(&imap), "r"(0), "r"(y0 + WR * warp), "r"(0), "r"(plane), "r"(x6_smem_u32(bar))
            : "memory");
    };
    if ((t & 31) == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(x6_smem_u32(bar)));
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        if ((int)blockIdx.x < ngroups) issue(blockIdx.x);
    }
    {
        const cx<T>* twg = static_cast<const cx<T>*>(a.tw);
        for (int e = t; e < M; e += 256) {
            tw[e] = twg[((e / R2) * (e % R2)) * (kTwiddleN / M)];
            tws[e] = twg[e * (kTwiddleN / (2 * M))];
        }
    }
    __syncthreads();
    // element k of this thread's row / slot s of the row's in-place exchange
    auto at = [&](int k) { return wbuf + ((k / L) * WR + (rl % WR)) * L + (k % L); };
    // with eight-element pieces the swizzled exchange addresses depend on the thread only through eight bases each (no
    // shift / xor per access); otherwise they are formed per access
    constexpr int NB = SW == 8 ? 8 : 1;
    cx<T>* wb[NB];      // element (tp ^ c) of the row's first pieces: the write of exchange row o1 lands o1 * R2 / L pieces further
    cx<T>* rbp[NB];     // element ((n & 7) ^ (tp & 7)) of exchange row tp: the read of column n adds its piece (n >> 3)
#pragma unroll
    for (int c = 0; c < NB; ++c) {
        wb[c] = at(tp ^ c);
        rbp[c] = at(tp * R2 + (c ^ (tp & 7)));
    }
    unsigned phase = 0;
    for (int grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
        {
            const unsigned addr = x6_smem_u32(bar);
            unsigned done;
            do {
                asm volatile(
                    "{\n"
                    ".reg .pred p;\n"
                    "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
                    "selp.u32 %0, 1, 0, p;\n"
                    "}\n"
                    : "=r"(done)
                    : "r"(addr), "r"(phase)
                    : "memory");
            } while (!done);
            phase ^= 1;
        }
        cx<T> v[R1];
        static_for<R1>([&](auto jc) {
            constexpr int j1 = decltype(jc)::value;
            const int k = tp + R2 * j1;
            const cx<T> Xk = *at(k), Xn = *at(M - k);
            const T ex = (T)0.5 * (Xk.x + Xn.x), ey = (T)0.5 * (Xk.y - Xn.y);
            const T dx = (T)0.5 * (Xk.x - Xn.x), dy = (T)0.5 * (Xk.y + Xn.y);
            const cx<T> w = tws[k];
            const T ox = dx * w.x + dy * w.y, oy = dy * w.x - dx * w.y;   // D * conj(w)
            v[j1] = {ex - oy, ey + ox};
        });
        Dif<T, +1, R1>::run(v);
        __syncwarp();                       // every thread of the row has read its inputs: the row's slots are free
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
                if constexpr (SW == 8) wb[o1 & 7][o1 * (R2 / L) * WR * L] = val;        // = *at(o1 * R2 + (tp ^ (o1 & 7)))
                else *at(o1 * R2 + (tp ^ (o1 & (SW - 1)))) = val;
            });
        });
        __syncwarp();
        cx<T> u[NT3][R2];
        static_for<NT3>([&](auto tc) {
            constexpr int it = decltype(tc)::value;
            const int o1 = tp + it * TPP;
            static_for<R2>([&](auto nc) {             // = *at(o1 * R2 + (n ^ (o1 & 7))), n = 8 (n >> 3) + (n & 7)
                constexpr int n = decltype(nc)::value;
                if constexpr (SW == 8) u[it][n] = rbp[n & 7][((n >> 3) + it * (TPP * R2 / L)) * WR * L];    // (tp + it TPP) & 7 == tp & 7
                else u[it][n] = *at(o1 * R2 + (n ^ (o1 & (SW - 1))));
            });
        });
        __syncwarp();                       // the rows of the warp are in registers: the warp's buffer is free
        if ((t & 31) == 0 && grp + (int)gridDim.x < ngroups) issue(grp + gridDim.x);
        int plane = grp / gpp;
        const int y0 = (grp - plane * gpp) * ROWS;
        if (a.pl_n) plane = (plane / a.pl_n) * a.pl_full + plane % a.pl_n;
        const int64_t row = (int64_t)plane * a.ny + y0 + rl;
        static_for<NT3>([&](auto tc) {
            constexpr int it = decltype(tc)::value;
            const int o1 = tp + it * TPP;
            Dif<T, +1, R2>::run(u[it]);
            cx<T>* dst = reinterpret_cast<cx<T>*>(out + row * a.real_rs) + o1;
            static_for<R2>([&](auto pc) {
                constexpr int p = decltype(pc)::value;
                constexpr int o2 = brev<R2>(p);
                if constexpr (!PRUNE || o2 < R2 / 2) {
                    if (!PRUNE || o1 + R1 * o2 < a.nc) dst[R1 * o2] = u[it][p];
                }
            });
        });
    }
}

// ------------------------------------------------------------------------------------------------------------------
// k6_xfwd: forward x pass without block barriers (Mc = R2 * R2: 256 in fp64 / fp32, 64 in fp64; zero-padded rows, any
// spectrum layout).  As in k2_xfwd the real rows of the block's next group are fetched into registers while the current
// group is transformed; as in k6_xinv a row's R2 threads sit in one warp and own the row's shared memory, so the exchange
// of the two-level transform (XOR swizzle within 128-byte pieces instead of a padding column), the natural-order copy and
// the split step need __syncwarp only.  Half spectra leave by per-thread stores straight from the split step.
// ------------------------------------------------------------------------------------------------------------------
template <typename T, int M>
__global__ void __launch_bounds__(256, 2) k6_xfwd(const T* __restrict__ in, cx<T>* __restrict__ out, X2Args a)
{
    using C = XCfg<M>;
    constexpr int R1 = C::R1, R2 = C::R2, TPP = C::TPP, ROWS = C::ROWS;
    constexpr int L = 128 / (int)sizeof(cx<T>);       // complex per 128-byte piece
    constexpr int SW = R2 < L ? R2 : L;               // the swizzle permutes within pieces (or within an exchange row)
    constexpr int NT3 = R1 / TPP;                     // second-step tasks (rows k1 = tp + it TPP of the exchange) per thread
    static_assert(R1 % TPP == 0 && R2 * (int)sizeof(cx<T>) >= 128 && (NT3 == 1 || TPP % 8 == 0), "an exchange row is whole pieces");
    cx<T>* tw = reinterpret_cast<cx<T>*>(fe2_smem);   // w_M^(n2 k1) at [k1 * R2 + n2]
    cx<T>* tws = tw + M;                              // w_2M^k, k < M
    cx<T>* buf = tws + M;                             // [ROWS][M]
    const int t = threadIdx.x, tp = t % TPP, rl = t / TPP;
    cx<T>* rb = buf + rl * M;
    constexpr int NLOAD = R1 / 2;
    const int64_t ngroups = (a.nrows + ROWS - 1) / ROWS;
    auto fetch = [&](int64_t grp, cx<T>* dst) {
        const int64_t row = grp * ROWS + rl;
        if (grp < ngroups && row < a.nrows) {
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
        for (int e = t; e < M; e += 256) {
            tw[e] = twg[((e / R2) * (e % R2)) * (kTwiddleN / M)];
            tws[e] = twg[e * (kTwiddleN / (2 * M))];
        }
    }
    __syncthreads();
    // exchange slot of element (k1, n2): k1 R2 + (n2 ^ (k1 & (SW - 1))).  With eight-element pieces the thread-dependent part
    // of both sides comes from eight bases; otherwise the addresses are formed per access
    constexpr int NB = SW == 8 ? 8 : 1;
    cx<T>* wb[NB];      // write side, thread n2 = tp:  rb + (tp ^ c), + k1 R2 with c = k1 & 7
    cx<T>* rd[NB];      // read side, thread k1 = tp:   rb + tp R2 + (c ^ (tp & 7)), + 8 (n2 >> 3) with c = n2 & 7
#pragma unroll
    for (int c = 0; c < NB; ++c) {
        wb[c] = rb + (tp ^ c);
        rd[c] = rb + tp * R2 + (c ^ (tp & 7));
    }
    for (int64_t grp = blockIdx.x; grp < ngroups; grp += gridDim.x) {
        const int64_t row = grp * ROWS + rl;
        const bool live = row < a.nrows;
        cx<T> v[R1];
        static_for<NLOAD>([&](auto ic) { v[decltype(ic)::value] = vn[decltype(ic)::value]; });
        fetch(grp + gridDim.x, vn);
        Dif<T, -1, R1, 0, true>::run(v);
        __syncwarp();                       // the split step of the previous group has read the row
        static_for<R1>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            constexpr int k1 = brev<R1>(p);
            cx<T> val = v[p];
            if constexpr (k1 != 0) val = cmul(val, tw[k1 * R2 + tp]);
            if constexpr (SW == 8) wb[k1 & 7][k1 * R2] = val;
            else rb[k1 * R2 + (tp ^ (k1 & (SW - 1)))] = val;
        });
        __syncwarp();
        cx<T> u[NT3][R2];
        static_for<NT3>([&](auto tc) {
            constexpr int it = decltype(tc)::value;
            static_for<R2>([&](auto nc) {
                constexpr int n = decltype(nc)::value;
                if constexpr (SW == 8) u[it][n] = rd[n & 7][8 * (n >> 3) + it * TPP * R2];     // (tp + it TPP) & 7 == tp & 7
                else u[it][n] = rb[(tp + it * TPP) * R2 + (n ^ ((tp + it * TPP) & (SW - 1)))];
            });
            Dif<T, -1, R2>::run(u[it]);
        });
        __syncwarp();                       // every thread of the row holds its exchange inputs
        static_for<NT3>([&](auto tc) {      // Z[k1 + R1 k2] in natural order
            constexpr int it = decltype(tc)::value;
            static_for<R2>([&](auto pc) {
                constexpr int p = decltype(pc)::value;
                rb[tp + it * TPP + R1 * brev<R2>(p)] = u[it][p];
            });
        });
        __syncwarp();
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
    }
}

template <typename T, int M>
static cudaError_t launch_xfwd6(const void* in, void* out, const X2Args& a, cudaStream_t st)
{
    using C = XCfg<M>;
    constexpr size_t smem = (size_t)(2 * M + C::ROWS * M) * sizeof(cx<T>);
    static PerDevice<int> cache;
    int& nblocks = cache.here();
    if (!nblocks) {
        cudaError_t e = cudaFuncSetAttribute(k6_xfwd<T, M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        int dev = 0, sms = 0, per = 0;
        if (e == cudaSuccess) e = cudaGetDevice(&dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, k6_xfwd<T, M>, 256, smem);
        if (e != cudaSuccess) return e;
        nblocks = sms * (per > 0 ? per : 1);
    }
    const int64_t ngroups = (a.nrows + C::ROWS - 1) / C::ROWS;
    const int grid = (int)(ngroups < nblocks ? ngroups : nblocks);
    k6_xfwd<T, M><<<grid, 256, smem, st>>>(static_cast<const T*>(in), static_cast<cx<T>*>(out), a);
    return cudaGetLastError();
}

// the barrier-free forward pass exists for Mc = 256 (fp64, fp32) and Mc = 128, 64 (fp64), zero-padded rows
template <typename T>
static bool try_launch_xfwd6(int M, const void* in, void* out, const X2Args& a, cudaError_t* err, cudaStream_t st)
{
    if (M == 256) {
        *err = launch_xfwd6<T, 256>(in, out, a, st);
        return true;
    }
    if constexpr (sizeof(T) == 8) {
        if (M == 64) {
            *err = launch_xfwd6<T, 64>(in, out, a, st);
            return true;
        }
        if (M == 128) {
            *err = launch_xfwd6<T, 128>(in, out, a, st);
            return true;
        }
    }
    return false;
}

// tensor map of the tiled half spectra S1[plane][g][y][L] (as reals) with the box of one row group; false if unavailable
template <typename T>
static bool make_x_map(const void* S1, int ny, int G, int nplanes, int rows, CUtensorMap* map)
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
    if (!enc || G > 256 || rows > 256) return false;
    const cuuint64_t dims[4] = {(cuuint64_t)(128 / sizeof(T)), (cuuint64_t)ny, (cuuint64_t)G, (cuuint64_t)nplanes};
    const cuuint64_t strides[3] = {128, (cuuint64_t)ny * 128, (cuuint64_t)G * ny * 128};
    const cuuint32_t box[4] = {(cuuint32_t)(128 / sizeof(T)), (cuuint32_t)rows, (cuuint32_t)G, 1};
    const cuuint32_t es[4] = {1, 1, 1, 1};
    return enc(map, sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4,
               const_cast<void*>(S1), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
               CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// persistent tensor-copy inverse pass when the layout is the tiled one (whole row groups per plane): Mc = 256 (fp64, fp32)
// and Mc = 128, 64 (fp64)
template <typename T, int M, bool PRUNE>
static bool launch_xinv6(const void* in, void* out, const X2Args& a, cudaError_t* err, cudaStream_t st)
{
    using C = XCfg<M>;
    constexpr int L = 128 / (int)sizeof(cx<T>);
    int lgL = 0;
    while ((1 << lgL) < L) ++lgL;
    if (a.lg != lgL || a.s_row != L || a.s_g != (int64_t)a.ny * L || a.ny % C::ROWS || a.s_plane % ((int64_t)a.ny * L)) return false;
    const int G = (int)(a.s_plane / ((int64_t)a.ny * L));
    if (a.nrows % a.ny || G * L < M + 1) return false;
    const int nplanes = (int)(a.nrows / a.ny);
    const int map_planes = a.pl_n ? nplanes / a.pl_n * a.pl_full : nplanes;
    CUtensorMap map;
    memset(&map, 0, sizeof(map));
    if (!make_x_map<T>(in, a.ny, G, map_planes, 32 / C::TPP, &map)) return false;       // one box = the rows of a warp
    const size_t smem = (size_t)G * C::ROWS * L * sizeof(cx<T>) + (size_t)2 * M * sizeof(cx<T>) + 8 * 8;
    if (smem > 113 * 1024) return false;
    static PerDevice<int> cache;
    int& sms = cache.here();
    if (!sms) {
        cudaError_t e = cudaFuncSetAttribute(k6_xinv<T, M, PRUNE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 113 * 1024);
        int dev = 0;
        if (e == cudaSuccess) e = cudaGetDevice(&dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) { sms = 0; *err = e; return true; }
    }
    // blocks per SM: depends on the shared-memory size, i.e. on the layout (G); asked again only when that changes
    struct Occ { size_t smem = 0; int per = 0; };
    static PerDevice<Occ> occ;
    Occ& o = occ.here();
    if (o.smem != smem) {
        int per = 0;
        if ((*err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, k6_xinv<T, M, PRUNE>, 256, smem)) != cudaSuccess) return true;
        o.smem = smem;
        o.per = per;
    }
    const int per = o.per;
    const int nblocks = sms * (per > 0 ? per : 1);
    const int ngroups = nplanes * (a.ny / C::ROWS);
    const int grid = ngroups < nblocks ? ngroups : nblocks;
    k6_xinv<T, M, PRUNE><<<grid, 256, smem, st>>>(static_cast<T*>(out), a, G, nplanes, map);
    *err = cudaGetLastError();
    return true;
}

template <typename T, bool PRUNE>
static bool try_launch_xinv6(int M, const void* in, void* out, const X2Args& a, cudaError_t* err, cudaStream_t st)
{
    if (M == 256) return launch_xinv6<T, 256, PRUNE>(in, out, a, err, st);
    if constexpr (sizeof(T) == 8) {
        if (M == 64) return launch_xinv6<T, 64, PRUNE>(in, out, a, err, st);
        if (M == 128) return launch_xinv6<T, 128, PRUNE>(in, out, a, err, st);
    }
    return false;
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
    if (prune) {
        cudaError_t e = cudaSuccess;
        if (v2::try_launch_xfwd6<T>(M, in, out, a, &e, st)) return e;
    }
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
    if (prune) {
        cudaError_t e = cudaSuccess;
        if (v2::try_launch_xinv6<T, true>(M, in, out, a, &e, st)) return e;
    }
    return v2::launch_x<T, false>(M, prune, in, out, a, st);
}

// planes [zb, zb + zn) of every one of the `comps` (= B * 3) components into planes [0, zn) of out[comps][nz][ny][n_real] -- the
// slab hand-over of FE_OPT_XL_SLABS.  Only the persistent tensor-copy kernel has the plane mapping: cudaErrorNotSupported elsewhere.
template <typename T>
cudaError_t launch_xinv2_slab(const FftCtx& c, const void* in, T* out, int n_real, int comps, int ny, int nz, int zb, int zn,
                              const int64_t spec[4], int lanes, cudaStream_t st)
{
    const int M = c.plan[0].M;
    if ((M != 256 && M != 128 && M != 64) || n_real > M || (n_real & 1)) return cudaErrorNotSupported;
    int lg = 0;
    while ((1 << lg) < lanes) ++lg;
    v2::X2Args a{c.tw, (int64_t)comps * zn * ny, n_real, (int)spec[0], lg, spec[1], spec[2], spec[3], n_real / 2, zn, nz, zb};
    cudaError_t e = cudaSuccess;
    if (v2::try_launch_xinv6<T, true>(M, in, out, a, &e, st)) return e;
    return cudaErrorNotSupported;
}
bool xinv_slab_supported(int Mc, int n_real, int ny, int lanes, size_t elem) { return elem == 8 && Mc == 256 && n_real <= Mc && ny % 16 == 0 && lanes == 8; }

template cudaError_t launch_xinv2_slab<double>(const FftCtx&, const void*, double*, int, int, int, int, int, int, const int64_t*, int, cudaStream_t);
template cudaError_t launch_xinv2_slab<float>(const FftCtx&, const void*, float*, int, int, int, int, int, int, const int64_t*, int, cudaStream_t);
template cudaError_t launch_xfwd2<double>(const FftCtx&, const double*, void*, int, int64_t, int64_t, const int64_t*, int, cudaStream_t);
template cudaError_t launch_xfwd2<float>(const FftCtx&, const float*, void*, int, int64_t, int64_t, const int64_t*, int, cudaStream_t);
template cudaError_t launch_xinv2<double>(const FftCtx&, const void*, double*, int, int64_t, int64_t, const int64_t*, int, cudaStream_t);
template cudaError_t launch_xinv2<float>(const FftCtx&, const void*, float*, int, int64_t, int64_t, const int64_t*, int, cudaStream_t);

}  // namespace fe
