// fe_tensor.cu -- a0: the cell-averaged dipolar interaction tensor on the circular padded box
// (Eq. 5-6 applied to cell-wise constant P, "similar to ...
// magnetostatics [40]" PAPER.md:115; readings A3 (what the tensor is) and A4 (periodic axes)).
//
//   N_ij(R) = -(1/(4 pi V)) int_cell d3r int_cell d3r' d_i d_j 1/|R + r - r'|
//
// evaluated in fp64 by two routes chosen per offset:
//   near  (gap < 3 cells): closed form, 4 pi V N_xx = -d2x d2y d2z f, 4 pi V N_xy = -d2x d2y d2z g with the
//         Newell-type primitives f, g and the 27-point second difference.  At this range the cancellation
//         inside the difference costs < 1e-14 absolute;
//   far   : Gauss-Legendre quadrature of the smooth equivalent form
//         N_ij(R) = -(1/(4 pi V)) int (dx-|u|)(dy-|v|)(dz-|w|) T_ij(R + (u,v,w)) du dv dw,
//         T_ij(rho) = 3 rho_i rho_j / rho^5 - delta_ij / rho^3, split at the kink of the triangle weight,
//         with 8/6/4/3/2 nodes per half interval depending on distance.  No cancellation at any range.
#include "fe_internal.h"
#include <math.h>

namespace fe {

constexpr int kTiers = 5;
__constant__ double c_glx[kTiers][8];
__constant__ double c_glw[kTiers][8];
__constant__ int c_gln[kTiers];
static const int h_gln[kTiers] = {8, 6, 4, 3, 2};

// Gauss-Legendre nodes on [-1, 1] by Newton iteration on P_n (host, long double).
static void gauss_legendre(int n, double* x, double* w)
{
    const long double pi = 3.141592653589793238462643383279502884L;
    for (int i = 0; i < n; ++i) {
        long double z = cosl(pi * (i + 0.75L) / (n + 0.5L)), pp = 1;
        for (int it = 0; it < 100; ++it) {
            long double p0 = 1, p1 = z;
            for (int k = 2; k <= n; ++k) {
                long double p2 = ((2 * k - 1) * z * p1 - (k - 1) * p0) / k;
                p0 = p1;
                p1 = p2;
            }
            pp = n * (z * p1 - p0) / (z * z - 1);
            long double dz = p1 / pp;
            z -= dz;
            if (fabsl(dz) < 1e-19L) break;
        }
        {
            long double p0 = 1, p1 = z;
            for (int k = 2; k <= n; ++k) {
                long double p2 = ((2 * k - 1) * z * p1 - (k - 1) * p0) / k;
                p0 = p1;
                p1 = p2;
            }
            pp = n * (z * p1 - p0) / (z * z - 1);
        }
        x[i] = (double)z;
        w[i] = (double)(2 / ((1 - z * z) * pp * pp));
    }
}

cudaError_t tensor_init_tables()
{
    double x[kTiers][8] = {}, w[kTiers][8] = {};
    for (int t = 0; t < kTiers; ++t) gauss_legendre(h_gln[t], x[t], w[t]);
    cudaError_t e;
    if ((e = cudaMemcpyToSymbol(c_glx, x, sizeof(x))) != cudaSuccess) return e;
    if ((e = cudaMemcpyToSymbol(c_glw, w, sizeof(w))) != cudaSuccess) return e;
    return cudaMemcpyToSymbol(c_gln, h_gln, sizeof(h_gln));
}

// ---- closed form ----------------------------------------------------------------------------------
__device__ double prim_f(double x, double y, double z)
{
    x = fabs(x); y = fabs(y); z = fabs(z);
    const double x2 = x * x, y2 = y * y, z2 = z * z, R = sqrt(x2 + y2 + z2);
    double r = 0.0;
    if (y != 0.0 && x2 + z2 != 0.0) r += 0.5 * y * (z2 - x2) * asinh(y / sqrt(x2 + z2));
    if (z != 0.0 && x2 + y2 != 0.0) r += 0.5 * z * (y2 - x2) * asinh(z / sqrt(x2 + y2));
    if (x != 0.0 && y != 0.0 && z != 0.0) r -= x * y * z * atan(y * z / (x * R));
    r += (2.0 * x2 - y2 - z2) * R / 6.0;
    return r;
}

__device__ double prim_g(double x, double y, double z)
{
    double sgn = 1.0;
    if (x < 0.0) { x = -x; sgn = -sgn; }
    if (y < 0.0) { y = -y; sgn = -sgn; }
    z = fabs(z);
    if (x == 0.0 || y == 0.0) return 0.0;
    const double x2 = x * x, y2 = y * y, z2 = z * z, R = sqrt(x2 + y2 + z2);
    double r = 0.0;
    if (z != 0.0) r += x * y * z * asinh(z / sqrt(x2 + y2));
    r += (y / 6.0) * (3.0 * z2 - y2) * asinh(x / sqrt(y2 + z2));
    r += (x / 6.0) * (3.0 * z2 - x2) * asinh(y / sqrt(x2 + z2));
    if (z != 0.0) {
        r -= (z * z2 / 6.0) * atan(x * y / (z * R));
        r -= 0.5 * z * y2 * atan(x * z / (y * R));
        r -= 0.5 * z * x2 * atan(y * z / (x * R));
    }
    r -= x * y * R / 3.0;
    return sgn * r;
}

__device__ double prim(int comp, double X, double Y, double Z)
{
    switch (comp) {
    case 0: return prim_f(X, Y, Z);
    case 1: return prim_f(Y, X, Z);
    case 2: return prim_f(Z, Y, X);
    case 3: return prim_g(X, Y, Z);
    case 4: return prim_g(X, Z, Y);
    default: return prim_g(Y, Z, X);
    }
}

__device__ void tensor_closed(const int* off, const double* d, double* out6)
{
    const double inv = -1.0 / (4.0 * 3.14159265358979323846 * d[0] * d[1] * d[2]);
    for (int comp = 0; comp < 6; ++comp) {
        double s = 0.0;
        for (int a = -1; a <= 1; ++a)
            for (int b = -1; b <= 1; ++b)
                for (int c = -1; c <= 1; ++c) {
                    const double wgt = (a == 0 ? -2.0 : 1.0) * (b == 0 ? -2.0 : 1.0) * (c == 0 ? -2.0 : 1.0);
                    s += wgt * prim(comp, (off[0] + a) * d[0], (off[1] + b) * d[1], (off[2] + c) * d[2]);
                }
        out6[comp] += s * inv;
    }
}

// ---- quadrature ------------------------------------------------------------------------------------
__device__ void tensor_quad(const int* off, const double* d, int tier, double* out6)
{
    const int n = c_gln[tier];
    const double X0 = off[0] * d[0], Y0 = off[1] * d[1], Z0 = off[2] * d[2];
    double sxx = 0, syy = 0, szz = 0, sxy = 0, sxz = 0, syz = 0;
    for (int iu = 0; iu < 2 * n; ++iu) {
        const int ju = iu < n ? iu : iu - n;
        const double tu = 0.5 * d[0] * (c_glx[tier][ju] + 1.0);            // in [0, dx]
        const double wu = 0.5 * d[0] * c_glw[tier][ju] * (d[0] - tu);
        const double X = X0 + (iu < n ? tu : -tu);
        for (int iv = 0; iv < 2 * n; ++iv) {
            const int jv = iv < n ? iv : iv - n;
            const double tv = 0.5 * d[1] * (c_glx[tier][jv] + 1.0);
            const double wuv = wu * 0.5 * d[1] * c_glw[tier][jv] * (d[1] - tv);
            const double Y = Y0 + (iv < n ? tv : -tv);
            for (int iw = 0; iw < 2 * n; ++iw) {
                const int jw = iw < n ? iw : iw - n;
                const double tz = 0.5 * d[2] * (c_glx[tier][jw] + 1.0);
                const double wt = wuv * 0.5 * d[2] * c_glw[tier][jw] * (d[2] - tz);
                const double Z = Z0 + (iw < n ? tz : -tz);
                const double r2 = X * X + Y * Y + Z * Z;
                const double ir = rsqrt(r2), ir2 = ir * ir;
                const double c3 = wt * ir * ir2;          // w / r^3
                const double c5 = 3.0 * c3 * ir2;         // 3 w / r^5
                sxx += c5 * X * X - c3;
                syy += c5 * Y * Y - c3;
                szz += c5 * Z * Z - c3;
                sxy += c5 * X * Y;
                sxz += c5 * X * Z;
                syz += c5 * Y * Z;
            }
        }
    }
    const double inv = -1.0 / (4.0 * 3.14159265358979323846 * d[0] * d[1] * d[2]);
    out6[0] += sxx * inv; out6[1] += syy * inv; out6[2] += szz * inv;
    out6[3] += sxy * inv; out6[4] += sxz * inv; out6[5] += syz * inv;
}

// N_ij at integer cell offset `off`, accumulated into out6 (xx yy zz xy xz yz)
__device__ void tensor_entry(const int* off, const double* d, double* out6)
{
    const double dmax = fmax(d[0], fmax(d[1], d[2]));
    double gap = 0.0;
    for (int a = 0; a < 3; ++a) gap = fmax(gap, (abs(off[a]) - 1) * d[a]);
    gap /= dmax;                        // clear distance between the two cells in units of the largest edge
    if (gap < 2.5) { tensor_closed(off, d, out6); return; }      // cubic cells: max |offset| <= 3
    const double dist = gap + 1.0;
    const int tier = dist < 6.0 ? 0 : dist < 12.0 ? 1 : dist < 32.0 ? 2 : dist < 128.0 ? 3 : 4;
    tensor_quad(off, d, tier, out6);
}

struct BoxArgs {
    int n[3], m[3], periodic[3], images[3];
    double d[3];
    int comp_first, ncomp;
};

// One thread per box entry.  Open axis (m >= 2 n): index t holds offset t (t < n), t - m (t > m - n), and 0 for
// n <= t <= m - n (never a pair offset).  Periodic axis: minimum image of t, the tie |d| = n/2 is the mean of both signs;
// K = sum over images q in [-R, R] of N(d + q n) (reading A4).
__global__ void k_tensor_box(double* __restrict__ box, BoxArgs a)
{
    const int64_t total = (int64_t)a.m[0] * a.m[1] * a.m[2];
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= total) return;
    const int t[3] = {(int)(e % a.m[0]), (int)((e / a.m[0]) % a.m[1]), (int)(e / ((int64_t)a.m[0] * a.m[1]))};
    int lo[3], cnt[3];
    bool unused = false;
    for (int ax = 0; ax < 3; ++ax) {
        const int n = a.n[ax];
        if (!a.periodic[ax]) {
            cnt[ax] = 1;
            if (t[ax] < n) lo[ax] = t[ax];
            else if (t[ax] <= a.m[ax] - n) { lo[ax] = 0; unused = true; }      // n .. m - n: never a pair offset
            else lo[ax] = t[ax] - a.m[ax];
        } else {
            if (2 * t[ax] < n) { lo[ax] = t[ax]; cnt[ax] = 1; }
            else if (2 * t[ax] > n) { lo[ax] = t[ax] - n; cnt[ax] = 1; }
            else { lo[ax] = -t[ax]; cnt[ax] = 2; }
        }
    }
    double acc[6] = {0, 0, 0, 0, 0, 0};
    if (!unused) {
        const int R0 = a.periodic[0] ? a.images[0] : 0, R1 = a.periodic[1] ? a.images[1] : 0,
                  R2 = a.periodic[2] ? a.images[2] : 0;
        for (int ux = 0; ux < cnt[0]; ++ux)
            for (int uy = 0; uy < cnt[1]; ++uy)
                for (int uz = 0; uz < cnt[2]; ++uz) {
                    const int d0[3] = {lo[0] + ux * a.n[0], lo[1] + uy * a.n[1], lo[2] + uz * a.n[2]};
                    for (int qx = -R0; qx <= R0; ++qx)
                        for (int qy = -R1; qy <= R1; ++qy)
                            for (int qz = -R2; qz <= R2; ++qz) {
                                const int off[3] = {d0[0] + qx * a.n[0], d0[1] + qy * a.n[1], d0[2] + qz * a.n[2]};
                                tensor_entry(off, a.d, acc);
                            }
                }
        const double nrm = 1.0 / (cnt[0] * cnt[1] * cnt[2]);
        for (int c = 0; c < 6; ++c) acc[c] *= nrm;
    }
    for (int c = 0; c < a.ncomp; ++c) box[(int64_t)c * total + e] = acc[a.comp_first + c];
}

cudaError_t launch_tensor_box(const Geometry& g, double* box, int comp_first, int ncomp, cudaStream_t st)
{
    BoxArgs a;
    for (int i = 0; i < 3; ++i) {
        a.n[i] = g.n[i]; a.m[i] = g.m[i]; a.periodic[i] = g.periodic[i]; a.images[i] = g.images[i];
        a.d[i] = g.d[i];
    }
    a.comp_first = comp_first;
    a.ncomp = ncomp;
    const int64_t total = (int64_t)g.m[0] * g.m[1] * g.m[2];
    k_tensor_box<<<(unsigned)((total + 127) / 128), 128, 0, st>>>(box, a);
    return cudaGetLastError();
}

// Zero-mode rule (reading A4): exactly two periodic axes, open axis w.  Every plane t_w != n_w of the
// box gets the constant that makes its sum equal 1 (component ww at offset 0) or 0 (everything else).
struct ZmArgs { int m[3]; int n[3]; int w; int is_ww; };

__global__ void k_zero_mode(double* __restrict__ box, ZmArgs a)
{
    __shared__ double red[256];
    const int tw = blockIdx.x;
    if (tw >= a.n[a.w] && tw <= a.m[a.w] - a.n[a.w]) return;      // unused planes of the padded open axis
    const int u = (a.w + 1) % 3, v = (a.w + 2) % 3;
    const int64_t stride[3] = {1, a.m[0], (int64_t)a.m[0] * a.m[1]};
    const int cnt = a.m[u] * a.m[v];
    double s = 0.0;
    for (int i = threadIdx.x; i < cnt; i += blockDim.x) {
        const int iu = i % a.m[u], iv = i / a.m[u];
        s += box[tw * stride[a.w] + iu * stride[u] + iv * stride[v]];
    }
    red[threadIdx.x] = s;
    __syncthreads();
    for (int h = blockDim.x / 2; h > 0; h >>= 1) {
        if ((int)threadIdx.x < h) red[threadIdx.x] += red[threadIdx.x + h];
        __syncthreads();
    }
    const double target = (a.is_ww && tw == 0) ? 1.0 : 0.0;
    const double c = (target - red[0]) / cnt;
    for (int i = threadIdx.x; i < cnt; i += blockDim.x) {
        const int iu = i % a.m[u], iv = i / a.m[u];
        box[tw * stride[a.w] + iu * stride[u] + iv * stride[v]] += c;
    }
}

// Fully periodic box (reading A4, last case): remove the mean of the image-summed table (k = 0 mode := 0).
__global__ void k_box_sum(const double* __restrict__ box, int64_t total, double* __restrict__ sum)
{
    __shared__ double red[256];
    double s = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) s += box[i];
    red[threadIdx.x] = s;
    __syncthreads();
    for (int h = blockDim.x / 2; h > 0; h >>= 1) {
        if ((int)threadIdx.x < h) red[threadIdx.x] += red[threadIdx.x + h];
        __syncthreads();
    }
    if (threadIdx.x == 0) atomicAdd(sum, red[0]);
}
__global__ void k_box_shift(double* __restrict__ box, int64_t total, const double* __restrict__ sum)
{
    const double mean = *sum / (double)total;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) box[i] -= mean;
}

cudaError_t launch_zero_mode(const Geometry& g, double* box, int comp, double* scratch, cudaStream_t st)
{
    const int np = g.periodic[0] + g.periodic[1] + g.periodic[2];
    if (g.zero_mode && np == 3) {
        const int64_t total = (int64_t)g.m[0] * g.m[1] * g.m[2];
        cudaError_t e = cudaMemsetAsync(scratch, 0, sizeof(double), st);
        if (e != cudaSuccess) return e;
        const int grid = (int)((total + 255) / 256 < 1184 ? (total + 255) / 256 : 1184);
        k_box_sum<<<grid, 256, 0, st>>>(box, total, scratch);
        k_box_shift<<<grid, 256, 0, st>>>(box, total, scratch);
        return cudaGetLastError();
    }
    if (!g.zero_mode || np != 2) return cudaSuccess;
    ZmArgs a;
    for (int i = 0; i < 3; ++i) { a.m[i] = g.m[i]; a.n[i] = g.n[i]; }
    a.w = !g.periodic[0] ? 0 : (!g.periodic[1] ? 1 : 2);
    a.is_ww = (comp == a.w);
    k_zero_mode<<<g.m[a.w], 256, 0, st>>>(box, a);
    return cudaGetLastError();
}

}  // namespace fe
