// fe_fft2.cuh -- register-resident two-level FFT building blocks of the size-specialised passes
// (Eq. 5-6).  Device code only; included by
// fe_fft2_axis.cu / fe_fft2_z.cu / fe_fft2_x.cu.  Nothing here is shared with oracle/.
//
// A transform of length M = R1 * R2 is computed as
//     X[k1 + R1 k2] = sum_{n2} w_R2^{n2 k2} [ w_M^{n2 k1} ( sum_{n1} x[n2 + R2 n1] w_R1^{n1 k1} ) ]
// step 1: one thread per n2 holds the R1 points x[n2 + R2 n1] in registers and runs an R1-point FFT,
// step 2: multiplies by the inter-step twiddle w_M^{n2 k1} (table in shared memory),
// exchange through shared memory (the only shared-memory round trip of the transform),
// step 3: one thread per k1 runs an R2-point FFT over n2.
// The register FFTs are radix-2 decimation-in-frequency recursions with compile-time twiddles (natural
// order in, bit-reversed out) and the mirrored decimation-in-time form (bit-reversed in, natural out).
// Zero-padded inputs skip the first butterfly stage (PRUNE); outputs that are not stored are removed by
// the compiler because every register index is a compile-time constant.
#pragma once
#include "fe_internal.h"
#include <utility>

namespace fe {
namespace v2 {

template <typename T> struct alignas(2 * sizeof(T)) cx { T x, y; };

template <typename T> __host__ __device__ __forceinline__ cx<T> cadd(cx<T> a, cx<T> b) { return {a.x + b.x, a.y + b.y}; }
template <typename T> __host__ __device__ __forceinline__ cx<T> csub(cx<T> a, cx<T> b) { return {a.x - b.x, a.y - b.y}; }
template <typename T> __host__ __device__ __forceinline__ cx<T> cmul(cx<T> a, cx<T> b)
{
    return {a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x};
}
template <typename T> __host__ __device__ __forceinline__ cx<T> cmulc(cx<T> a, cx<T> b)   // a * conj(b)
{
    return {a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y};
}
// a * w (DIR < 0) or a * conj(w) (DIR > 0), w from the forward-sign table
template <typename T, int DIR> __host__ __device__ __forceinline__ cx<T> cmuld(cx<T> a, cx<T> w)
{
    return DIR < 0 ? cmul(a, w) : cmulc(a, w);
}

template <int... I, typename F>
__host__ __device__ __forceinline__ void static_for_impl(F&& f, std::integer_sequence<int, I...>)
{
    (f(std::integral_constant<int, I>{}), ...);
}
// f(integral_constant<int, 0>) ... f(integral_constant<int, N-1>): every index is a compile-time constant
template <int N, typename F> __host__ __device__ __forceinline__ void static_for(F&& f)
{
    static_for_impl(f, std::make_integer_sequence<int, N>{});
}

// bit reversal of p within log2(R) bits
template <int R> __host__ __device__ constexpr int brev(int p)
{
    int r = 0;
    for (int b = 1; b < R; b <<= 1) {
        r = (r << 1) | (p & 1);
        p >>= 1;
    }
    return r;
}

// cos(pi i / 16), sin(pi i / 16), i = 0..8
__host__ __device__ constexpr double cos16(int i)
{
    switch (i) {
        case 0: return 1.0;
        case 1: return 0.9807852804032304491262;
        case 2: return 0.9238795325112867561282;
        case 3: return 0.8314696123025452370788;
        case 4: return 0.7071067811865475244008;
        case 5: return 0.5555702330196022247428;
        case 6: return 0.3826834323650897717285;
        case 7: return 0.1950903220161282678483;
        default: return 0.0;
    }
}
__host__ __device__ constexpr double sin16(int i) { return cos16(8 - i); }

// a * exp(DIR * 2 pi i * IDX / 32), 0 <= IDX < 16
template <typename T, int DIR, int IDX> __host__ __device__ __forceinline__ cx<T> mulw32(cx<T> a)
{
    constexpr T s = (T)DIR;
    if constexpr (IDX == 0) {
        return a;
    } else if constexpr (IDX == 8) {
        return {-s * a.y, s * a.x};
    } else if constexpr (IDX == 4) {
        constexpr T h = (T)0.7071067811865475244008;
        return {h * (a.x - s * a.y), h * (a.y + s * a.x)};
    } else if constexpr (IDX == 12) {
        constexpr T h = (T)0.7071067811865475244008;
        return {-h * (a.x + s * a.y), h * (s * a.x - a.y)};
    } else {
        constexpr T c = (T)(IDX <= 8 ? cos16(IDX) : -cos16(16 - IDX));
        constexpr T sn = (T)((double)DIR * (IDX <= 8 ? sin16(IDX) : sin16(16 - IDX)));
        return {c * a.x - sn * a.y, c * a.y + sn * a.x};
    }
}

// in-register decimation in frequency on v[OFF .. OFF+LEN): natural order in, v[OFF + p] = X[brev<LEN>(p)] out.
// PRUNE: the upper half of the input is zero (first stage needs no additions).
template <typename T, int DIR, int LEN, int OFF = 0, bool PRUNE = false> struct Dif {
    static __host__ __device__ __forceinline__ void run(cx<T>* v)
    {
        constexpr int H = LEN / 2;
        static_for<H>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            const cx<T> a = v[OFF + i];
            if constexpr (PRUNE) {
                v[OFF + i + H] = mulw32<T, DIR, i * (32 / LEN)>(a);
            } else {
                const cx<T> b = v[OFF + i + H];
                v[OFF + i] = cadd(a, b);
                v[OFF + i + H] = mulw32<T, DIR, i * (32 / LEN)>(csub(a, b));
            }
        });
        if constexpr (LEN > 2) {
            Dif<T, DIR, H, OFF, false>::run(v);
            Dif<T, DIR, H, OFF + H, false>::run(v);
        }
    }
};
template <typename T, int DIR, int OFF, bool PRUNE> struct Dif<T, DIR, 1, OFF, PRUNE> {
    static __host__ __device__ __forceinline__ void run(cx<T>*) {}
};

// in-register decimation in time: v[OFF + p] = X[brev<LEN>(p)] in, natural order out
template <typename T, int DIR, int LEN, int OFF = 0> struct Dit {
    static __host__ __device__ __forceinline__ void run(cx<T>* v)
    {
        constexpr int H = LEN / 2;
        if constexpr (LEN > 2) {
            Dit<T, DIR, H, OFF>::run(v);
            Dit<T, DIR, H, OFF + H>::run(v);
        }
        static_for<H>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            const cx<T> a = v[OFF + i];
            const cx<T> b = mulw32<T, DIR, i * (32 / LEN)>(v[OFF + i + H]);
            v[OFF + i] = cadd(a, b);
            v[OFF + i + H] = csub(a, b);
        });
    }
};
template <typename T, int DIR, int OFF> struct Dit<T, DIR, 1, OFF> {
    static __host__ __device__ __forceinline__ void run(cx<T>*) {}
};

// ---- fused multiply-add butterflies (decimation in time) ----------------------------------------------------
// a' = a + w b, b' = a - w b with w = exp(DIR * 2 pi i * IDX / 32), 0 <= IDX < 16.  For a general w = c + i s the
// product is folded into the additions: with t = s / c (|c| >= |s|), b~ = (b.x - t b.y, b.y + t b.x) and
// a +- w b = a +- c b~, six fused multiply-adds instead of the four multiplies and four additions of the plain
// form; when |s| > |c| the roles of c and s are exchanged (w b = s (u b.x - b.y, u b.y + b.x), u = c / s) so that
// the ratio never exceeds one.  HI = false drops b' (pruned output).
__host__ __device__ __forceinline__ constexpr double cabs_c(double v) { return v < 0 ? -v : v; }
template <typename T, int DIR, int IDX, bool HI = true>
__host__ __device__ __forceinline__ void bfly_dit(cx<T>& a, cx<T>& b)
{
    if constexpr (IDX == 0) {
        const cx<T> t = b;
        if constexpr (HI) b = csub(a, t);
        a = cadd(a, t);
    } else if constexpr (IDX == 8) {                         // w = DIR * i
        const cx<T> t = DIR > 0 ? cx<T>{-b.y, b.x} : cx<T>{b.y, -b.x};
        if constexpr (HI) b = csub(a, t);
        a = cadd(a, t);
    } else {
        constexpr double c = IDX <= 8 ? cos16(IDX) : -cos16(16 - IDX);
        constexpr double s = (double)DIR * (IDX <= 8 ? sin16(IDX) : sin16(16 - IDX));
        T br, bi, m;
        if constexpr (cabs_c(c) >= cabs_c(s)) {
            constexpr T t = (T)(s / c);
            br = fma(-t, b.y, b.x);
            bi = fma(t, b.x, b.y);
            m = (T)c;
        } else {
            constexpr T u = (T)(c / s);
            br = fma(u, b.x, -b.y);
            bi = fma(u, b.y, b.x);
            m = (T)s;
        }
        if constexpr (HI) b = {fma(-m, br, a.x), fma(-m, bi, a.y)};
        a = {fma(m, br, a.x), fma(m, bi, a.y)};
    }
}

// in-register decimation in time with the fused butterflies: v[OFF + p] = x[brev<LEN>(p)] in, v[OFF + k] = X[k] out.
// PIN: x[n] = 0 for n >= LEN/2 (the odd positions p are never read); POUT: only X[k], k < LEN/2, are produced.
template <typename T, int DIR, int LEN, int OFF = 0, bool PIN = false, bool POUT = false> struct DitF {
    static __host__ __device__ __forceinline__ void run(cx<T>* v)
    {
        constexpr int H = LEN / 2;
        if constexpr (LEN == 2 && PIN) {
            v[OFF + 1] = v[OFF];
        } else {
            if constexpr (LEN > 2) {
                DitF<T, DIR, H, OFF, PIN, false>::run(v);
                DitF<T, DIR, H, OFF + H, PIN, false>::run(v);
            }
            static_for<H>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                bfly_dit<T, DIR, i * (32 / LEN), !POUT>(v[OFF + i], v[OFF + i + H]);
            });
        }
    }
};
template <typename T, int DIR, int OFF, bool PIN, bool POUT> struct DitF<T, DIR, 1, OFF, PIN, POUT> {
    static __host__ __device__ __forceinline__ void run(cx<T>*) {}
};

// factorisation M = R1 * R2 (R1 >= R2) of the supported lengths
template <int M> struct Fact;
template <> struct Fact<64> { static constexpr int R1 = 8, R2 = 8; };
template <> struct Fact<128> { static constexpr int R1 = 16, R2 = 8; };
template <> struct Fact<256> { static constexpr int R1 = 16, R2 = 16; };
template <> struct Fact<512> { static constexpr int R1 = 32, R2 = 16; };

// fill the forward-sign inter-step table tw[e] = exp(-2 pi i e / M), e < M, from the global 2048-entry table
template <typename T, int M>
__device__ __forceinline__ void load_twiddles(cx<T>* tw, const cx<T>* __restrict__ twg, int tid, int nthreads)
{
    constexpr int mul = kTwiddleN / M;
    for (int e = tid; e < M; e += nthreads) tw[e] = twg[e * mul];
}

extern __shared__ __align__(16) unsigned char fe2_smem[];

}  // namespace v2
}  // namespace fe
