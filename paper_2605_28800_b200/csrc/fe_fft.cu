// fe_fft.cu -- hand-written batched power-of-two FFT passes for the electrostatic convolution
// ("electrostatic field ... FFT", Eq. 5-6).
//
// Design:
//  * every pass keeps a tile of pencils in shared memory: [position along the transformed axis][lane],
//    lanes = 128 bytes of consecutive kx (or 8 rows for the x passes), so global traffic is whole
//    128-byte lines and shared-memory traffic is conflict free;
//  * forward transforms are in-place decimation-in-frequency (natural in, digit-reversed out), inverse
//    transforms are the mirrored decimation-in-time (digit-reversed in, natural out): no reordering pass.
//    The digit-reversed positions are mapped to natural frequency rows when a tile is stored, which is free
//    because rows are independent 128-byte segments;
//  * zero padding is never materialised: the padded half is zero-filled in shared memory on load and the
//    discarded half is simply not stored (pruned transforms);
//  * the z transform, the 6-component symmetric tensor multiply and the inverse z transform are one kernel
//    (k_zmul), the padded z extent never reaches HBM;
//  * x is the real axis: R2C/C2R through a half-length complex FFT plus the split/merge step.
#include "fe_internal.h"

namespace fe {

template <typename T> struct alignas(2 * sizeof(T)) cx { T x, y; };

template <typename T> __device__ __forceinline__ cx<T> cadd(cx<T> a, cx<T> b) { return {a.x + b.x, a.y + b.y}; }
template <typename T> __device__ __forceinline__ cx<T> csub(cx<T> a, cx<T> b) { return {a.x - b.x, a.y - b.y}; }
template <typename T> __device__ __forceinline__ cx<T> cmul(cx<T> a, cx<T> b)
{
    return {a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x};
}
// a * conj(b)
template <typename T> __device__ __forceinline__ cx<T> cmulc(cx<T> a, cx<T> b)
{
    return {a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y};
}
// multiply by -i (forward, DIR < 0) or +i (inverse)
template <typename T, int DIR> __device__ __forceinline__ cx<T> rot90(cx<T> a)
{
    return DIR < 0 ? cx<T>{a.y, -a.x} : cx<T>{-a.y, a.x};
}

// R-point DFT, natural order in and out: v[q'] = sum_q v[q] exp(DIR * 2 pi i q q' / R)
template <typename T, int R, int DIR> struct Bfly;

template <typename T, int DIR> struct Bfly<T, 2, DIR> {
    static __device__ __forceinline__ void run(cx<T>* v)
    {
        cx<T> a = v[0], b = v[1];
        v[0] = cadd(a, b);
        v[1] = csub(a, b);
    }
};

template <typename T, int DIR> struct Bfly<T, 4, DIR> {
    static __device__ __forceinline__ void run(cx<T>* v)
    {
        cx<T> t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
        cx<T> t2 = cadd(v[1], v[3]), t3 = rot90<T, DIR>(csub(v[1], v[3]));
        v[0] = cadd(t0, t2);
        v[1] = cadd(t1, t3);
        v[2] = csub(t0, t2);
        v[3] = csub(t1, t3);
    }
};

template <typename T, int DIR> struct Bfly<T, 8, DIR> {
    static __device__ __forceinline__ void run(cx<T>* v)
    {
        cx<T> e[4] = {v[0], v[2], v[4], v[6]};
        cx<T> o[4] = {v[1], v[3], v[5], v[7]};
        Bfly<T, 4, DIR>::run(e);
        Bfly<T, 4, DIR>::run(o);
        const T h = (T)0.70710678118654752440;
        cx<T> o1, o3;
        if (DIR < 0) {   // w8 = (1 - i)/sqrt2, w8^3 = (-1 - i)/sqrt2
            o1 = {(o[1].x + o[1].y) * h, (o[1].y - o[1].x) * h};
            o3 = {(o[3].y - o[3].x) * h, -(o[3].x + o[3].y) * h};
        } else {         // conj
            o1 = {(o[1].x - o[1].y) * h, (o[1].x + o[1].y) * h};
            o3 = {-(o[3].x + o[3].y) * h, (o[3].x - o[3].y) * h};
        }
        cx<T> o2 = rot90<T, DIR>(o[2]);
        v[0] = cadd(e[0], o[0]);
        v[4] = csub(e[0], o[0]);
        v[1] = cadd(e[1], o1);
        v[5] = csub(e[1], o1);
        v[2] = cadd(e[2], o2);
        v[6] = csub(e[2], o2);
        v[3] = cadd(e[3], o3);
        v[7] = csub(e[3], o3);
    }
};

// One radix-R stage over `ntiles` tiles of pencils held in shared memory.
//   element (tile t, position x, lane l) lives at s[t * tile_stride + x * pitch + l]
//   forward (DIR < 0): v = DFT_R(inputs at base + q * Ls/R), output q' multiplied by w_Ls^(j q')
//   inverse (DIR > 0): the exact inverse of that stage up to the factor R
template <typename T, int R, int DIR>
__device__ __forceinline__ void fft_stage(cx<T>* s, int pitch, int logLanes, int ntiles, int tile_stride,
                                          int M, int Ls, const cx<T>* __restrict__ tw)
{
    const int sub = Ls / R;
    const int logsub = 31 - __clz(sub);
    const int nbf = M / R;
    const int lognbf = 31 - __clz(nbf);
    const int lanes = 1 << logLanes;
    const int total = (nbf << logLanes) * ntiles;
    const int twmul = kTwiddleN / Ls;
    const int step = sub * pitch;
    for (int i = threadIdx.x; i < total; i += blockDim.x) {
        const int lane = i & (lanes - 1);
        int b = i >> logLanes;
        const int t = b >> lognbf;
        b &= nbf - 1;
        const int j = b & (sub - 1);
        const int g = b >> logsub;
        cx<T>* p = s + (size_t)t * tile_stride + (g * Ls + j) * pitch + lane;
        cx<T> v[R];
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = p[q * step];
        if (DIR < 0) {
            Bfly<T, R, DIR>::run(v);
            if (sub > 1) {
#pragma unroll
                for (int q = 1; q < R; ++q) v[q] = cmul(v[q], tw[j * q * twmul]);
            }
        } else {
            if (sub > 1) {
#pragma unroll
                for (int q = 1; q < R; ++q) v[q] = cmulc(v[q], tw[j * q * twmul]);
            }
            Bfly<T, R, DIR>::run(v);
        }
#pragma unroll
        for (int q = 0; q < R; ++q) p[q * step] = v[q];
    }
}

template <typename T, int DIR>
__device__ __forceinline__ void fft_stage_any(int R, cx<T>* s, int pitch, int logLanes, int ntiles,
                                              int tile_stride, int M, int Ls, const cx<T>* __restrict__ tw)
{
    if (R == 8) fft_stage<T, 8, DIR>(s, pitch, logLanes, ntiles, tile_stride, M, Ls, tw);
    else if (R == 4) fft_stage<T, 4, DIR>(s, pitch, logLanes, ntiles, tile_stride, M, Ls, tw);
    else fft_stage<T, 2, DIR>(s, pitch, logLanes, ntiles, tile_stride, M, Ls, tw);
}

// All stages of one transform; block-wide, synchronises before the first and after the last stage.
template <typename T, int DIR>
__device__ __forceinline__ void fft_tiles(cx<T>* s, int pitch, int logLanes, int ntiles, int tile_stride,
                                          const AxisPlan& pl, const cx<T>* __restrict__ tw)
{
    if (DIR < 0) {
        int Ls = pl.M;
        for (int st = 0; st < pl.nst; ++st) {
            __syncthreads();
            fft_stage_any<T, DIR>(pl.radix[st], s, pitch, logLanes, ntiles, tile_stride, pl.M, Ls, tw);
            Ls /= pl.radix[st];
        }
    } else {
        int Ls = 1;
        for (int st = pl.nst - 1; st >= 0; --st) {
            Ls *= pl.radix[st];
            __syncthreads();
            fft_stage_any<T, DIR>(pl.radix[st], s, pitch, logLanes, ntiles, tile_stride, pl.M, Ls, tw);
        }
    }
    __syncthreads();
}

extern __shared__ __align__(16) unsigned char fe_smem[];

// ------------------------------------------------------------------------------------------------
// x passes: 8 rows per block, shared layout [position][row] with pitch 9 (conflict free both when the
// rows are loaded along x and when the butterflies run across rows).
// ------------------------------------------------------------------------------------------------
constexpr int kRowsX = 8;
constexpr int kPitchX = kRowsX + 1;

struct XArgs {
    AxisPlan plan;
    const uint16_t* invperm;
    const void* tw;
    int n_real;            // valid reals per row on the real side (n_in forward, n_out inverse), even
    int rows;              // rows per slab
    int64_t real_rs, real_ss, spec_rs, spec_ss;
};

// real row x[0..n_real) (zero beyond) of padded length m = 2 Mc  ->  X[k], k = 0..Mc.
//   z[j] = x[2j] + i x[2j+1], Z = FFT_Mc(z);  Xe = (Z[k] + conj Z[Mc-k])/2, Xo = -i (Z[k] - conj Z[Mc-k])/2,
//   X[k] = Xe + w_m^k Xo.
template <typename T>
__global__ void __launch_bounds__(kThreads) k_xfwd(const T* __restrict__ in, cx<T>* __restrict__ out, XArgs a)
{
    cx<T>* s = reinterpret_cast<cx<T>*>(fe_smem);
    const cx<T>* tw = static_cast<const cx<T>*>(a.tw);
    const int Mc = a.plan.M, logM = a.plan.logM;
    const int row0 = blockIdx.y * kRowsX;
    const int nrow = min(kRowsX, a.rows - row0);
    const int nc = a.n_real >> 1;
    const T* ib = in + (int64_t)blockIdx.x * a.real_ss + (int64_t)row0 * a.real_rs;
    for (int idx = threadIdx.x; idx < kRowsX * Mc; idx += blockDim.x) {
        const int r = idx >> logM, j = idx & (Mc - 1);
        cx<T> v = {0, 0};
        if (r < nrow && j < nc) v = *reinterpret_cast<const cx<T>*>(ib + r * a.real_rs + 2 * j);
        s[j * kPitchX + r] = v;
    }
    fft_tiles<T, -1>(s, kPitchX, 3, 1, 0, a.plan, tw);
    cx<T>* ob = out + (int64_t)blockIdx.x * a.spec_ss + (int64_t)row0 * a.spec_rs;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
    const int twm = kTwiddleN / (2 * Mc);
    for (int r = warp; r < nrow; r += nwarp)
        for (int k = lane; k <= Mc; k += 32) {
            const cx<T> Zk = s[a.invperm[k & (Mc - 1)] * kPitchX + r];
            const cx<T> Zn = s[a.invperm[(Mc - k) & (Mc - 1)] * kPitchX + r];
            const T ex = (T)0.5 * (Zk.x + Zn.x), ey = (T)0.5 * (Zk.y - Zn.y);
            const T ox = (T)0.5 * (Zk.y + Zn.y), oy = (T)-0.5 * (Zk.x - Zn.x);
            const cx<T> w = tw[k * twm];
            ob[r * a.spec_rs + k] = {ex + ox * w.x - oy * w.y, ey + ox * w.y + oy * w.x};
        }
}

// X[k], k = 0..Mc  ->  first n_real reals of the (unnormalised, factor Mc) inverse real transform.
template <typename T>
__global__ void __launch_bounds__(kThreads) k_xinv(const cx<T>* __restrict__ in, T* __restrict__ out, XArgs a)
{
    cx<T>* s = reinterpret_cast<cx<T>*>(fe_smem);
    const cx<T>* tw = static_cast<const cx<T>*>(a.tw);
    const int Mc = a.plan.M;
    const int row0 = blockIdx.y * kRowsX;
    const int nrow = min(kRowsX, a.rows - row0);
    const cx<T>* ib = in + (int64_t)blockIdx.x * a.spec_ss + (int64_t)row0 * a.spec_rs;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
    const int twm = kTwiddleN / (2 * Mc);
    for (int r = warp; r < kRowsX; r += nwarp)
        for (int k = lane; k < Mc; k += 32) {
            cx<T> Z = {0, 0};
            if (r < nrow) {
                const cx<T> Xk = ib[r * a.spec_rs + k], Xn = ib[r * a.spec_rs + Mc - k];
                const T ex = (T)0.5 * (Xk.x + Xn.x), ey = (T)0.5 * (Xk.y - Xn.y);
                const T dx = (T)0.5 * (Xk.x - Xn.x), dy = (T)0.5 * (Xk.y + Xn.y);
                const cx<T> w = tw[k * twm];
                const T ox = dx * w.x + dy * w.y, oy = dy * w.x - dx * w.y;   // D * conj(w)
                Z = {ex - oy, ey + ox};
            }
            s[a.invperm[k] * kPitchX + r] = Z;
        }
    fft_tiles<T, +1>(s, kPitchX, 3, 1, 0, a.plan, tw);
    const int nc = a.n_real >> 1;            // any value up to Mc (open axes need not be powers of two)
    T* ob = out + (int64_t)blockIdx.x * a.real_ss + (int64_t)row0 * a.real_rs;
    for (int idx = threadIdx.x; idx < kRowsX * nc; idx += blockDim.x) {
        const int r = idx / nc, j = idx - r * nc;
        if (r < nrow) *reinterpret_cast<cx<T>*>(ob + r * a.real_rs + 2 * j) = s[j * kPitchX + r];
    }
}

// ------------------------------------------------------------------------------------------------
// strided pass along y (or z): tile [M][lanes], lanes consecutive kx.
// ------------------------------------------------------------------------------------------------
struct AxisArgs {
    AxisPlan plan;
    const uint16_t* perm;
    const void* tw;
    int n_keep;
    int logLanes;
    int64_t in_sa, in_so, in_sb, out_sa, out_so, out_sb;
};

template <typename T, int DIR>
__global__ void __launch_bounds__(kThreads) k_axis(const cx<T>* __restrict__ in, cx<T>* __restrict__ out, AxisArgs a)
{
    cx<T>* s = reinterpret_cast<cx<T>*>(fe_smem);
    const cx<T>* tw = static_cast<const cx<T>*>(a.tw);
    const int M = a.plan.M, logLanes = a.logLanes, lanes = 1 << logLanes;
    const int kx0 = blockIdx.x << logLanes;
    const cx<T>* ib = in + (int64_t)blockIdx.z * a.in_sb + (int64_t)blockIdx.y * a.in_so + kx0;
    cx<T>* ob = out + (int64_t)blockIdx.z * a.out_sb + (int64_t)blockIdx.y * a.out_so + kx0;
    const int total = M << logLanes;
    if (DIR < 0) {
        for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
            const int r = idx >> logLanes, lane = idx & (lanes - 1);
            cx<T> v = {0, 0};
            if (r < a.n_keep) v = ib[(int64_t)r * a.in_sa + lane];
            s[idx] = v;
        }
        fft_tiles<T, DIR>(s, lanes, logLanes, 1, 0, a.plan, tw);
        for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
            const int p = idx >> logLanes, lane = idx & (lanes - 1);
            ob[(int64_t)a.perm[p] * a.out_sa + lane] = s[idx];
        }
    } else {
        for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
            const int p = idx >> logLanes, lane = idx & (lanes - 1);
            s[idx] = ib[(int64_t)a.perm[p] * a.in_sa + lane];
        }
        fft_tiles<T, DIR>(s, lanes, logLanes, 1, 0, a.plan, tw);
        for (int idx = threadIdx.x; idx < (a.n_keep << logLanes); idx += blockDim.x) {
            const int r = idx >> logLanes, lane = idx & (lanes - 1);
            ob[(int64_t)r * a.out_sa + lane] = s[idx];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// fused z pass: forward z transform of the three components, E~_i = -escale * sum_j K~_ij P~_j
// (Eq. 5-6 in k-space; K~ real, symmetric, stored for kz <= Mz/2, ky <= My/2 with the sign rules of
// its parity: xy odd in y, xz odd in z, yz odd in y and z), inverse z transform, first nz outputs kept.
// ------------------------------------------------------------------------------------------------
struct ZArgs {
    AxisPlan plan;
    const uint16_t* perm;
    const void* tw;
    const DevMember* members;
    int nz, My, logLanes, pitch;
};

template <typename T>
__global__ void __launch_bounds__(kThreads) k_zmul(cx<T>* __restrict__ S, const T* __restrict__ Kt, ZArgs a)
{
    cx<T>* s = reinterpret_cast<cx<T>*>(fe_smem);
    const cx<T>* tw = static_cast<const cx<T>*>(a.tw);
    const int M = a.plan.M, logM = a.plan.logM, logLanes = a.logLanes, lanes = 1 << logLanes;
    const int kx0 = blockIdx.x << logLanes, ky = blockIdx.y, b = blockIdx.z;
    const int64_t sa = (int64_t)a.My * a.pitch, cs = (int64_t)a.nz * sa;
    cx<T>* base = S + (int64_t)b * 3 * cs + (int64_t)ky * a.pitch + kx0;
    const int tile = M << logLanes;
    for (int idx = threadIdx.x; idx < 3 * tile; idx += blockDim.x) {
        const int c = idx >> (logM + logLanes), rem = idx & (tile - 1);
        const int r = rem >> logLanes, lane = rem & (lanes - 1);
        cx<T> v = {0, 0};
        if (r < a.nz) v = base[c * cs + r * sa + lane];
        s[idx] = v;
    }
    fft_tiles<T, -1>(s, lanes, logLanes, 3, tile, a.plan, tw);
    {
        const int Hy = a.My / 2 + 1, Hz = M / 2 + 1;
        const int kym = ky <= a.My / 2 ? ky : a.My - ky;
        const T sy = ky > a.My / 2 ? (T)-1 : (T)1;
        const int64_t kcs = (int64_t)Hz * Hy * a.pitch;
        const T esc = (T)(-a.members[b].escale);
        for (int idx = threadIdx.x; idx < tile; idx += blockDim.x) {
            const int p = idx >> logLanes, lane = idx & (lanes - 1);
            const int kz = a.perm[p];
            const int kzm = kz <= M / 2 ? kz : M - kz;
            const T sz = kz > M / 2 ? (T)-1 : (T)1;
            const T* kp = Kt + ((int64_t)kzm * Hy + kym) * a.pitch + kx0 + lane;
            const T Kxx = __ldg(kp), Kyy = __ldg(kp + kcs), Kzz = __ldg(kp + 2 * kcs);
            const T Kxy = sy * __ldg(kp + 3 * kcs), Kxz = sz * __ldg(kp + 4 * kcs);
            const T Kyz = sy * sz * __ldg(kp + 5 * kcs);
            const cx<T> Px = s[idx], Py = s[idx + tile], Pz = s[idx + 2 * tile];
            s[idx] = {esc * (Kxx * Px.x + Kxy * Py.x + Kxz * Pz.x), esc * (Kxx * Px.y + Kxy * Py.y + Kxz * Pz.y)};
            s[idx + tile] = {esc * (Kxy * Px.x + Kyy * Py.x + Kyz * Pz.x),
                             esc * (Kxy * Px.y + Kyy * Py.y + Kyz * Pz.y)};
            s[idx + 2 * tile] = {esc * (Kxz * Px.x + Kyz * Py.x + Kzz * Pz.x),
                                 esc * (Kxz * Px.y + Kyz * Py.y + Kzz * Pz.y)};
        }
    }
    fft_tiles<T, +1>(s, lanes, logLanes, 3, tile, a.plan, tw);
    const int keep = a.nz << logLanes;
    for (int idx = threadIdx.x; idx < 3 * keep; idx += blockDim.x) {
        const int c = idx / keep, rem = idx - c * keep;
        const int r = rem >> logLanes, lane = rem & (lanes - 1);
        base[c * cs + r * sa + lane] = s[c * tile + rem];
    }
}

// complex fp64 spectrum of one tensor component on the box -> real table for kz <= Mz/2, ky <= My/2.
// Entry (kz, ky, kx) is written at kz * k_skz + ky * k_sky + (kx >> lg) * k_sg + (kx & (2^lg - 1)): row-major
// (k_skz = Hy pitch, k_sky = pitch, k_sg = 2^lg) or the tiled layout of fe_api.cu.
template <typename T>
__global__ void k_extract(const cx<double>* __restrict__ Sbox, T* __restrict__ Kt, int My, int Lx, int pitch64,
                          int pitchT, double scale, int lg, int64_t k_skz, int64_t k_sky, int64_t k_sg)
{
    const int kz = blockIdx.z, ky = blockIdx.y;
    for (int kx = blockIdx.x * blockDim.x + threadIdx.x; kx < pitchT; kx += gridDim.x * blockDim.x) {
        double v = 0.0;
        if (kx < Lx) v = Sbox[((int64_t)kz * My + ky) * pitch64 + kx].x * scale;
        Kt[(int64_t)kz * k_skz + (int64_t)ky * k_sky + (int64_t)(kx >> lg) * k_sg + (kx & ((1 << lg) - 1))] = (T)v;
    }
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
static int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }

template <typename T>
cudaError_t launch_xfwd(const FftCtx& c, const T* in, void* out, int n_in, int rows_per_slab, int slabs,
                        int64_t in_row_stride, int64_t in_slab_stride, int64_t out_row_stride,
                        int64_t out_slab_stride, cudaStream_t st)
{
    XArgs a{c.plan[0], c.tab[0].invperm, c.tw, n_in, rows_per_slab, in_row_stride, in_slab_stride,
            out_row_stride, out_slab_stride};
    dim3 grid(slabs, (rows_per_slab + kRowsX - 1) / kRowsX, 1);
    size_t smem = (size_t)c.plan[0].M * kPitchX * sizeof(cx<T>);
    k_xfwd<T><<<grid, kThreads, smem, st>>>(in, static_cast<cx<T>*>(out), a);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_xinv(const FftCtx& c, const void* in, T* out, int n_out, int rows_per_slab, int slabs,
                        int64_t in_row_stride, int64_t in_slab_stride, int64_t out_row_stride,
                        int64_t out_slab_stride, cudaStream_t st)
{
    XArgs a{c.plan[0], c.tab[0].invperm, c.tw, n_out, rows_per_slab, out_row_stride, out_slab_stride,
            in_row_stride, in_slab_stride};
    dim3 grid(slabs, (rows_per_slab + kRowsX - 1) / kRowsX, 1);
    size_t smem = (size_t)c.plan[0].M * kPitchX * sizeof(cx<T>);
    k_xinv<T><<<grid, kThreads, smem, st>>>(static_cast<const cx<T>*>(in), out, a);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_axis(const FftCtx& c, int axis, int dir, const void* in, void* out, int n_keep, int lanes,
                        int pitch_used, int outer, int batch, int64_t in_sa, int64_t in_so, int64_t in_sb,
                        int64_t out_sa, int64_t out_so, int64_t out_sb, cudaStream_t st)
{
    AxisArgs a{c.plan[axis], c.tab[axis].perm, c.tw, n_keep, ilog2(lanes), in_sa, in_so, in_sb,
               out_sa, out_so, out_sb};
    dim3 grid(pitch_used / lanes, outer, batch);
    size_t smem = (size_t)c.plan[axis].M * lanes * sizeof(cx<T>);
    if (dir < 0)
        k_axis<T, -1><<<grid, kThreads, smem, st>>>(static_cast<const cx<T>*>(in), static_cast<cx<T>*>(out), a);
    else
        k_axis<T, +1><<<grid, kThreads, smem, st>>>(static_cast<const cx<T>*>(in), static_cast<cx<T>*>(out), a);
    return cudaGetLastError();
}

size_t zmul_smem_bytes(int Mz, int lanes, size_t cx_bytes) { return (size_t)3 * Mz * lanes * cx_bytes; }

template <typename T>
cudaError_t launch_zmul(const FftCtx& c, void* S, const T* Kt, const DevMember* members, int nz, int My,
                        int lanes, int pitch, int batch, cudaStream_t st)
{
    ZArgs a{c.plan[2], c.tab[2].perm, c.tw, members, nz, My, ilog2(lanes), pitch};
    dim3 grid(pitch / lanes, My, batch);
    size_t smem = zmul_smem_bytes(c.plan[2].M, lanes, sizeof(cx<T>));
    k_zmul<T><<<grid, kThreads, smem, st>>>(static_cast<cx<T>*>(S), Kt, a);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_extract(const void* Sbox, T* Kt_comp, int Mz, int My, int Lx, int pitch64, int pitchT,
                           double scale, int lanes, int64_t k_skz, int64_t k_sky, int64_t k_sg, cudaStream_t st)
{
    const int Hz = Mz / 2 + 1, Hy = My / 2 + 1;
    int lg = 0;
    while ((1 << lg) < lanes) ++lg;
    dim3 grid((pitchT + 127) / 128, Hy, Hz);
    k_extract<T><<<grid, 128, 0, st>>>(static_cast<const cx<double>*>(Sbox), Kt_comp, My, Lx, pitch64, pitchT, scale,
                                       lg, k_skz, k_sky, k_sg);
    return cudaGetLastError();
}

cudaError_t fft_configure()
{
    const int lim = 227 * 1024;
    cudaError_t e;
#define FE_SET(k) if ((e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, lim)) != cudaSuccess) return e
    FE_SET(k_xfwd<double>); FE_SET(k_xfwd<float>);
    FE_SET(k_xinv<double>); FE_SET(k_xinv<float>);
    FE_SET((k_axis<double, -1>)); FE_SET((k_axis<double, 1>));
    FE_SET((k_axis<float, -1>)); FE_SET((k_axis<float, 1>));
    FE_SET(k_zmul<double>); FE_SET(k_zmul<float>);
#undef FE_SET
    return cudaSuccess;
}

#define FE_INST(T)                                                                                                 \
    template cudaError_t launch_xfwd<T>(const FftCtx&, const T*, void*, int, int, int, int64_t, int64_t, int64_t,  \
                                        int64_t, cudaStream_t);                                                    \
    template cudaError_t launch_xinv<T>(const FftCtx&, const void*, T*, int, int, int, int64_t, int64_t, int64_t,  \
                                        int64_t, cudaStream_t);                                                    \
    template cudaError_t launch_axis<T>(const FftCtx&, int, int, const void*, void*, int, int, int, int, int,      \
                                        int64_t, int64_t, int64_t, int64_t, int64_t, int64_t, cudaStream_t);       \
    template cudaError_t launch_zmul<T>(const FftCtx&, void*, const T*, const DevMember*, int, int, int, int, int, \
                                        cudaStream_t);                                                             \
    template cudaError_t launch_extract<T>(const void*, T*, int, int, int, int, int, double, int, int64_t, int64_t,   \
                                           int64_t, cudaStream_t);
FE_INST(double)
FE_INST(float)

}  // namespace fe
