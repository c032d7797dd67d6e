// fe_local.cu -- a4/a5: fused local step, and a6: energy reduction.
//   k = L * active * (E_Land + E_Grad + E_Elec + E_Ext)                      PAPER.md:33 (Eq. 1)
//   E_Land = -d f_Land/dP, f_Land of Eq. 3 with per-axis a1 and four 8th-order slots
//   E_Grad = exact gradient of the discrete Eq. 4 energy (reading A2):
//            sum_a c_ia [P_i(r+e_a) - 2 P_i(r) + P_i(r-e_a)] / D_a^2   (bond missing -> that difference is 0)
//          + Gm sum_{j != i} [D_j P_j (r+e_i) - D_j P_j (r-e_i)] / (2 D_i), D_j = centred difference with
//            zero outside the sample / in vacuum cells, c_ia = G11 (a == i) or G44 + G44', Gm = G12 + G44 - G44'
//   then the integrator stage:  Yout = baseY + cy * k,  accOut = accIn + ca * k
#include "fe_internal.h"
#include <string.h>
#include <type_traits>
#include <cuda.h>          // CUtensorMap and cuTensorMapEncodeTiled's signature only; the entry point is fetched at run time

namespace fe {

template <typename T> struct LandauT {
    T a1x, a1y, a1z, a11, a12, a111, a112, a123, a1111, a1112, a1122, a1123;
    __device__ explicit LandauT(const DevLandau& m)
        : a1x((T)m.a1[0]), a1y((T)m.a1[1]), a1z((T)m.a1[2]), a11((T)m.a11), a12((T)m.a12), a111((T)m.a111),
          a112((T)m.a112), a123((T)m.a123), a1111((T)m.a1111), a1112((T)m.a1112), a1122((T)m.a1122),
          a1123((T)m.a1123) {}
    // d f / d P_i / P_i with (a, b, c) = (P_i^2, other two squared)
    __device__ __forceinline__ T dfd(T a1i, T a, T b, T c) const
    {
        const T bc = b + c, b2c2 = b * b + c * c, bxc = b * c;
        T s = (T)2 * a1i + (T)4 * a11 * a + (T)2 * a12 * bc + (T)6 * a111 * a * a;
        s += a112 * ((T)4 * a * bc + (T)2 * b2c2) + (T)2 * a123 * bxc;
        s += (T)8 * a1111 * a * a * a + a1112 * ((T)6 * a * a * bc + (T)2 * (b * b * b + c * c * c));
        s += (T)4 * a1122 * a * b2c2 + a1123 * ((T)4 * a * bxc + (T)2 * bxc * bc);
        return s;
    }
    __device__ __forceinline__ T f(T a, T b, T c) const
    {
        T r = a1x * a + a1y * b + a1z * c + a11 * (a * a + b * b + c * c) + a12 * (a * b + b * c + c * a);
        r += a111 * (a * a * a + b * b * b + c * c * c);
        r += a112 * (a * a * (b + c) + b * b * (a + c) + c * c * (a + b)) + a123 * a * b * c;
        r += a1111 * (a * a * a * a + b * b * b * b + c * c * c * c);
        r += a1112 * (a * a * a * (b + c) + b * b * b * (a + c) + c * c * c * (a + b));
        r += a1122 * (a * a * b * b + b * b * c * c + c * c * a * a) + a1123 * a * b * c * (a + b + c);
        return r;
    }
};

// Coefficients of -E_Land,i / P_i = d f_Land / d P_i / P_i (Eq. 3) with the integer factors folded in:
//   k1_i + k11 a + k12 (b+c) + k111 a^2 + k112 [2 a (b+c) + b^2 + c^2] + k123 b c
//   + k1111 a^3 + k1112 [3 a^2 (b+c) + b^3 + c^3] + k1122 a (b^2+c^2) + k1123 b c (2 a + b + c)
// with (a, b, c) = (P_i^2, the other two squared).
template <typename T> struct LandauD {
    T k1x, k1y, k1z, k11, k12, k111, k112, k123, k1111, k1112, k1122, k1123;
    int o8;       // any 8th-order slot non-zero
    int active;
    __device__ LandauD() {}
    __device__ explicit LandauD(const DevLandau& m)
        : k1x((T)(2 * m.a1[0])), k1y((T)(2 * m.a1[1])), k1z((T)(2 * m.a1[2])), k11((T)(4 * m.a11)), k12((T)(2 * m.a12)),
          k111((T)(6 * m.a111)), k112((T)(2 * m.a112)), k123((T)(2 * m.a123)), k1111((T)(8 * m.a1111)),
          k1112((T)(2 * m.a1112)), k1122((T)(4 * m.a1122)), k1123((T)(2 * m.a1123)),
          o8(m.a1111 != 0.0 || m.a1112 != 0.0 || m.a1122 != 0.0 || m.a1123 != 0.0), active(m.active != 0) {}
    // a2 = a^2, b2c2 = b^2 + c^2, bc = b + c, bxc = b c
    __device__ __forceinline__ T dfd(T k1i, T a, T a2, T bc, T b2c2, T bxc, T b3c3) const
    {
        T s = k1i + k11 * a;
        s += k12 * bc;
        s += k111 * a2;
        s += k112 * ((a + a) * bc + b2c2);
        s += k123 * bxc;
        if (o8) {
            s += k1111 * (a2 * a);
            s += k1112 * ((T)3 * a2 * bc + b3c3);
            s += k1122 * (a * b2c2);
            s += k1123 * (bxc * (a + a + bc));
        }
        return s;
    }
};

// neighbour coordinate along one axis; returns -1 if it falls outside an open axis
__device__ __forceinline__ int nb(int c, int s, int n, int per)
{
    int v = c + s;
    if (v < 0) return per ? v + n : -1;
    if (v >= n) return per ? v - n : -1;
    return v;
}

template <typename T, bool MAP>
struct Grid {
    const T* p[3];
    const uint8_t* map;
    const DevLandau* mats;
    int nx, ny, nz;
    // value of component c at (x,y,z): 0 outside or in a vacuum cell; *ok tells whether the cell exists
    __device__ __forceinline__ T val(int c, int x, int y, int z, bool& ok) const
    {
        if ((x | y | z) < 0) { ok = false; return (T)0; }
        const int64_t r = ((int64_t)z * ny + y) * nx + x;
        if (!mats[MAP ? map[r] : 0].active) { ok = false; return (T)0; }     // (no map: every cell is material 0)
        ok = true;
        return p[c][r];
    }
    __device__ __forceinline__ T val(int c, int x, int y, int z) const
    {
        bool ok;
        return val(c, x, y, z, ok);
    }
};

// ------------------------------------------------------------------------------------------------
// k_local: one block owns a 32 x 8 column of cells and marches along z.  The three components of the
// current plane and its two z neighbours live in a 4-slot ring of shared-memory tiles with a one-cell halo
// (zero outside the sample / in vacuum cells, wrapped on periodic axes) plus one validity byte per cell, so
// every P value is fetched from global memory once per block and all 7 / 19 stencil taps come from shared
// memory.  One __syncthreads per plane: the plane z+1 is loaded into the slot that held z-3.
// ------------------------------------------------------------------------------------------------
constexpr int kTX = 32, kTY = 8, kHX = kTX + 2, kHY = kTY + 2, kTile = kHX * kHY;   // 34 x 10 = 340
constexpr int kNL = (3 * kTile + 255) / 256;                                        // loader entries per thread

template <typename T, bool MAP, bool MIXED>
__global__ void __launch_bounds__(256, 2) k_local(LocalArgs a)
{
    extern __shared__ __align__(16) unsigned char lsm[];
    T* tiles = reinterpret_cast<T*>(lsm);                                   // [4][3][kTile]
    unsigned char* flags = lsm + (size_t)4 * 3 * kTile * sizeof(T);         // [4][kTile]
    LandauD<T>* smats = reinterpret_cast<LandauD<T>*>(flags + 4 * kTile + 8);  // [nmat]  (offset is 8-aligned)
    unsigned char* sact = reinterpret_cast<unsigned char*>(smats + a.nmat);  // [nmat]

    const int nx = a.n[0], ny = a.n[1], nz = a.n[2];
    const int ntx = (nx + kTX - 1) / kTX;
    const int x0 = (blockIdx.x % ntx) * kTX, y0 = (blockIdx.x / ntx) * kTY;
    const int z0 = a.zbeg + blockIdx.y * a.zchunk, z1 = min(z0 + a.zchunk, a.zend);
    const int b = blockIdx.z;
    const int t = threadIdx.x, tx = t & 31, ty = t >> 5;
    const int64_t nxy = (int64_t)nx * ny, N = nxy * nz;
    const T* Y = static_cast<const T*>(a.Y) + (int64_t)b * 3 * N;
    const DevLandau* mats = a.mats + (int64_t)b * a.nmat;
    for (int m = t; m < a.nmat; m += 256) {
        smats[m] = LandauD<T>(mats[m]);
        sact[m] = mats[m].active != 0;
    }
    const DevMember mem = a.members[b];

    // loader entries: shared offset, in-plane global offset (-1: outside an open axis), component
    int l_so[kNL], l_go[kNL];
    const T* l_ptr[kNL];
#pragma unroll
    for (int k = 0; k < kNL; ++k) {
        const int idx = t + 256 * k;
        l_so[k] = -1;
        l_go[k] = -1;
        l_ptr[k] = Y;
        if (idx < 3 * kTile) {
            const int rem = idx % kTile, yy = rem / kHX, xx = rem % kHX;
            int gx = x0 - 1 + xx, gy = y0 - 1 + yy;
            bool in = true;
            if (gx < 0 || gx >= nx) { if (a.periodic[0]) gx = ((gx % nx) + nx) % nx; else in = false; }
            if (gy < 0 || gy >= ny) { if (a.periodic[1]) gy = ((gy % ny) + ny) % ny; else in = false; }
            l_so[k] = idx;
            l_go[k] = in ? gy * nx + gx : -1;
            if (in) l_ptr[k] = Y + (int64_t)(idx / kTile) * N + l_go[k];
        }
    }
    // global -> registers (issued one plane ahead of its use), registers -> shared tile
    T pre[kNL];
    bool pok[kNL];
    auto fetch_plane = [&](int z) {
        int zz = z;
        bool zin = true;
        if (zz < 0 || zz >= nz) { if (a.periodic[2]) zz = ((zz % nz) + nz) % nz; else zin = false; }
        const int64_t r0 = (int64_t)zz * nxy;
#pragma unroll
        for (int k = 0; k < kNL; ++k) {
            const bool ok = zin && l_go[k] >= 0;
            pre[k] = ok ? l_ptr[k][r0] : (T)0;
            pok[k] = ok;
            if (MAP) { if (ok) pok[k] = sact[a.map[r0 + l_go[k]]] != 0; }
        }
    };
    auto store_plane = [&](int z) {
        const int slot = z & 3;
        T* tl = tiles + slot * 3 * kTile;
        unsigned char* fl = flags + slot * kTile;
#pragma unroll
        for (int k = 0; k < kNL; ++k) {
            if (l_so[k] < 0) continue;
            tl[l_so[k]] = pok[k] ? pre[k] : (T)0;
            if (MAP && l_so[k] < kTile) fl[l_so[k]] = pok[k];
        }
    };
    __syncthreads();          // coefficient tables visible (fetch_plane reads sact)
    fetch_plane(z0 - 1);
    store_plane(z0 - 1);
    fetch_plane(z0);
    store_plane(z0);
    fetch_plane(z0 + 1);

    const int x = x0 + tx, y = y0 + ty;
    const bool inside = x < nx && y < ny;
    const int64_t rxy = (int64_t)y * nx + x;
    const int c0 = (ty + 1) * kHX + tx + 1;
    // without a material map the existence of a neighbour is pure geometry
    const T gxf = (T)((x > 0 || a.periodic[0]) + (x < nx - 1 || a.periodic[0]));
    const T gyf = (T)((y > 0 || a.periodic[1]) + (y < ny - 1 || a.periodic[1]));
    const T G11 = (T)mem.G11, Gt = (T)mem.Gt, Gm = (T)mem.Gm, L = (T)mem.L;
    const T ix = (T)a.id2[0], iy = (T)a.id2[1], iz = (T)a.id2[2];
    const T qxy = Gm * (T)a.i4[0], qxz = Gm * (T)a.i4[1], qyz = Gm * (T)a.i4[2];
    const T cy = (T)a.cy, ca = (T)a.ca;
    const double wv = mem.wave ? sin(mem.womega * a.t + mem.wphase) : 0.0;      // E_ext sampled at the stage time
    const T ex0 = (T)(mem.Eext[0] + mem.wamp[0] * wv), ex1 = (T)(mem.Eext[1] + mem.wamp[1] * wv),
            ex2 = (T)(mem.Eext[2] + mem.wamp[2] * wv);
    const T* Ee = (a.terms & 4u) && a.Eelec ? static_cast<const T*>(a.Eelec) + (int64_t)b * 3 * N : nullptr;
    const T* base = a.baseY ? static_cast<const T*>(a.baseY) + (int64_t)b * 3 * N : nullptr;
    const bool base_is_Y = a.baseY == a.Y;
    T* Yout = static_cast<T*>(a.Yout) + (int64_t)b * 3 * N;
    const T* ai = a.accOut ? static_cast<const T*>(a.accIn) + (int64_t)b * 3 * N : nullptr;
    T* ao = a.accOut ? static_cast<T*>(a.accOut) + (int64_t)b * 3 * N : nullptr;
    const LandauD<T> lc0 = smats[0];

    T en[3] = {0, 0, 0};
    if (Ee && inside) {
        const int64_t r = (int64_t)z0 * nxy + rxy;
        en[0] = Ee[r]; en[1] = Ee[N + r]; en[2] = Ee[2 * N + r];
    }
    for (int z = z0; z < z1; ++z) {
        store_plane(z + 1);
        __syncthreads();
        if (z + 1 < z1) fetch_plane(z + 2);      // in flight while plane z is computed
        if (!inside) continue;
        const T ec[3] = {en[0], en[1], en[2]};
        if (Ee && z + 1 < z1) {
            const int64_t rn = (int64_t)(z + 1) * nxy + rxy;
            en[0] = Ee[rn]; en[1] = Ee[N + rn]; en[2] = Ee[2 * N + rn];
        }
        const T* m0 = tiles + ((z - 1) & 3) * 3 * kTile;      // plane z-1
        const T* c = tiles + (z & 3) * 3 * kTile;             // plane z
        const T* p1 = tiles + ((z + 1) & 3) * 3 * kTile;      // plane z+1
        const unsigned char* fm = flags + ((z - 1) & 3) * kTile;
        const unsigned char* fc = flags + (z & 3) * kTile;
        const unsigned char* fp = flags + ((z + 1) & 3) * kTile;
        const int64_t r = (int64_t)z * nxy + rxy;
        T k[3] = {0, 0, 0};
        const bool act = MAP ? fc[c0] != 0 : lc0.active != 0;       // without a map every cell is material 0 (vacuum: pinned)
        if (act) {
            const T px = c[c0], py = c[kTile + c0], pz = c[2 * kTile + c0];
            T E0 = 0, E1 = 0, E2 = 0;
            if (a.terms & 1u) {
                const LandauD<T> lc = MAP ? smats[a.map[r]] : lc0;
                const T A = px * px, B = py * py, C = pz * pz;
                const T A2 = A * A, B2 = B * B, C2 = C * C;
                T A3 = 0, B3 = 0, C3 = 0;
                if (lc.o8) { A3 = A2 * A; B3 = B2 * B; C3 = C2 * C; }
                E0 -= px * lc.dfd(lc.k1x, A, A2, B + C, B2 + C2, B * C, B3 + C3);
                E1 -= py * lc.dfd(lc.k1y, B, B2, C + A, C2 + A2, C * A, C3 + A3);
                E2 -= pz * lc.dfd(lc.k1z, C, C2, A + B, A2 + B2, A * B, A3 + B3);
            }
            if (a.terms & 2u) {
                // bonds: sum over existing neighbours of c_ia / D_a^2 (P_i(nb) - P_i(r)); a missing neighbour holds 0
                const T nxf = MAP ? (T)(fc[c0 - 1] + fc[c0 + 1]) : gxf;
                const T nyf = MAP ? (T)(fc[c0 - kHX] + fc[c0 + kHX]) : gyf;
                const T nzf = MAP ? (T)(fm[c0] + fp[c0])
                                  : (T)((z > 0 || a.periodic[2]) + (z < nz - 1 || a.periodic[2]));
#pragma unroll
                for (int i = 0; i < 3; ++i) {
                    const T* ci = c + i * kTile;
                    const T p = ci[c0];
                    const T sx = ci[c0 - 1] + ci[c0 + 1] - nxf * p;
                    const T sy = ci[c0 - kHX] + ci[c0 + kHX] - nyf * p;
                    const T sz = m0[i * kTile + c0] + p1[i * kTile + c0] - nzf * p;
                    const T e = (i == 0 ? G11 : Gt) * ix * sx + (i == 1 ? G11 : Gt) * iy * sy + (i == 2 ? G11 : Gt) * iz * sz;
                    if (i == 0) E0 += e; else if (i == 1) E1 += e; else E2 += e;
                }
                if (MIXED) {
                    // Gm sum_{j != i} [P_j(+i+j) - P_j(+i-j) - P_j(-i+j) + P_j(-i-j)] / (4 D_i D_j)
                    const T* cx_ = c;               // Px plane z
                    const T* cy_ = c + kTile;       // Py
                    const T* cz_ = c + 2 * kTile;   // Pz
                    const T dxy_y = cy_[c0 + 1 + kHX] - cy_[c0 + 1 - kHX] - cy_[c0 - 1 + kHX] + cy_[c0 - 1 - kHX];
                    const T dxy_x = cx_[c0 + 1 + kHX] - cx_[c0 + 1 - kHX] - cx_[c0 - 1 + kHX] + cx_[c0 - 1 - kHX];
                    const T dxz_z = p1[2 * kTile + c0 + 1] - m0[2 * kTile + c0 + 1] - p1[2 * kTile + c0 - 1] + m0[2 * kTile + c0 - 1];
                    const T dxz_x = p1[c0 + 1] - m0[c0 + 1] - p1[c0 - 1] + m0[c0 - 1];
                    const T dyz_z = p1[2 * kTile + c0 + kHX] - m0[2 * kTile + c0 + kHX] - p1[2 * kTile + c0 - kHX] + m0[2 * kTile + c0 - kHX];
                    const T dyz_y = p1[kTile + c0 + kHX] - m0[kTile + c0 + kHX] - p1[kTile + c0 - kHX] + m0[kTile + c0 - kHX];
                    E0 += qxy * dxy_y + qxz * dxz_z;
                    E1 += qxy * dxy_x + qyz * dyz_z;
                    E2 += qxz * dxz_x + qyz * dyz_y;
                }
            }
            if (Ee) { E0 += ec[0]; E1 += ec[1]; E2 += ec[2]; }
            if (a.terms & 8u) { E0 += ex0; E1 += ex1; E2 += ex2; }
            k[0] = L * E0; k[1] = L * E1; k[2] = L * E2;
        }
        T bv[3] = {0, 0, 0};
        if (base) {
            if (base_is_Y) {
                // the stage base is the state itself (Euler): take it from the tile; vacuum cells hold their raw value
                if (act) { bv[0] = c[c0]; bv[1] = c[kTile + c0]; bv[2] = c[2 * kTile + c0]; }
                else { bv[0] = base[r]; bv[1] = base[N + r]; bv[2] = base[2 * N + r]; }
            } else {
                bv[0] = base[r]; bv[1] = base[N + r]; bv[2] = base[2 * N + r];
            }
        }
        if (a.kOut) {
            T* ko = static_cast<T*>(a.kOut) + (int64_t)b * 3 * N;
#pragma unroll
            for (int i = 0; i < 3; ++i) ko[i * N + r] = k[i];
        }
        for (int j = 0; j < a.nlin; ++j) {
            const T* lkj = static_cast<const T*>(a.lk[j]) + (int64_t)b * 3 * N;
            const T cj = (T)a.lc[j];
#pragma unroll
            for (int i = 0; i < 3; ++i) bv[i] = bv[i] + cj * lkj[i * N + r];
        }
#pragma unroll
        for (int i = 0; i < 3; ++i) Yout[i * N + r] = bv[i] + cy * k[i];
        if (ao) {
#pragma unroll
            for (int i = 0; i < 3; ++i) ao[i * N + r] = ai[i * N + r] + ca * k[i];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// k_local2: the same z-marching scheme with a 64 x 8 column per block and TWO x-adjacent cells per thread.
// Interior cell x of the tile sits at column 2 + x of a 68-wide shared row, so the pair (2 tx, 2 tx + 1) is a
// 16-byte (fp64) aligned vector: centre, y and z taps of both cells come with one vector load each, which
// halves the shared-memory instructions per cell; the plane loader moves pairs as well.
// ------------------------------------------------------------------------------------------------
constexpr int k2TX = 64, k2PX = 68, k2HY = kTY + 2, k2Tile = k2PX * k2HY;        // 68 x 10 = 680
constexpr int k2Pairs = k2HY * (k2TX / 2);                                      // pair entries per component
constexpr int k2Sing = k2HY * 2;                                                // halo-column entries per component
constexpr int k2NL = (3 * (k2Pairs + k2Sing) + 255) / 256;                      // loader entries per thread (4)

template <typename T> struct alignas(2 * sizeof(T)) pair_t { T a, b; };

// cp.async of BYTES (4, 8 or 16) with zero fill: src_bytes = 0 writes zeros without touching global memory
template <int BYTES> __device__ __forceinline__ void cp_async_zfill(void* smem, const void* gmem, int src_bytes)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2, %3;\n" ::"r"(s), "l"(gmem), "n"(BYTES), "r"(src_bytes));
}

// mbarrier / tensor-copy helpers of the TMA halo loader
__device__ __forceinline__ unsigned lsm_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void l_mbar_init(void* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(lsm_u32(bar)), "r"(count));
}
__device__ __forceinline__ void l_mbar_expect_tx(void* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(lsm_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void l_mbar_arrive(void* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(lsm_u32(bar)) : "memory");
}
__device__ __forceinline__ void l_mbar_wait(void* bar, unsigned parity)
{
    const unsigned addr = lsm_u32(bar);
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
// 4-D box (x, y, z, component) of the state -> shared memory; coordinates outside the tensor read as zero
__device__ __forceinline__ void l_tma_load_4d(void* smem_dst, const CUtensorMap* map, int cx0, int cy0, int cz0, int cc0, void* bar)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];\n" ::"r"(
            lsm_u32(smem_dst)),
        "l"(map), "r"(cx0), "r"(cy0), "r"(cz0), "r"(cc0), "r"(lsm_u32(bar))
        : "memory");
}

// bytes of one plane slot of k_local2 (three components of a 68 x 10 tile), rounded up to the 128-byte alignment of a
// tensor copy's destination
template <typename T, bool WIDE = false> __host__ __device__ constexpr size_t k2_slot_bytes()
{
    return ((size_t)3 * (WIDE ? 72 : k2PX) * k2HY * sizeof(T) + 127) / 128 * 128;
}

// TMA = true (no material map, no periodic axis): a plane of the halo tile arrives as ONE tensor copy
// (cp.async.bulk.tensor, box 68 x 10 x 1 x 3 components starting at (x0 - 2, y0 - 1, z); cells outside the sample are
// zero-filled by the copy engine) issued by one thread and completed on an mbarrier, instead of four cp.async per thread.
// EPI != 0: a stage of forward Euler / Heun / classical RK4 with all four terms (terms == FE_TERM_ALL with E_elec, a stage
// base, no folded stage combination, no raw-k output) -- the runtime switches of the epilogue become compile-time constants,
// which frees the registers their pointers and flags hold and with them the per-plane recomputation of loop invariants:
//   EPI 1: baseY == Y, no accumulator (Euler);  2: baseY == Y, accumulator (first stage of Heun / RK4);
//   EPI 3: baseY != Y, no accumulator (last stage of Heun / RK4);  4: baseY != Y, accumulator (RK4 stages 2 and 3);
//   EPI 5: baseY == Y, raw k written, two folded terms (AB3M2 predictor with history);  6: baseY != Y, one folded term
//   (AB3M2 corrector);  7: no base, no accumulator: the plain right-hand side of fe_rhs.
// EPI 0 is the general epilogue (fe_rhs, RK45, the first AB3M2 steps, partial term sets).
// VAC = true (general epilogue without a map only): material 0 of some member is vacuum, i.e. the whole member is pinned;
// every other instantiation without a map takes all cells as active.
template <typename T, bool MAP, bool MIXED, bool TMA = false, int EPI = 0, bool VAC = false>
__global__ void __launch_bounds__(256, 2) k_local2(LocalArgs a, const __grid_constant__ CUtensorMap tmap)
{
    static_assert(!VAC || (!MAP && EPI == 0), "the vacuum check belongs to the general epilogue without a map");
    constexpr bool PLAIN = EPI != 0;                 // specialised epilogue
    constexpr bool BASEY = EPI == 1 || EPI == 2 || EPI == 5, ACC = EPI == 2 || EPI == 4, KOUT = EPI == 5;
    constexpr int NLIN = EPI == 5 ? 2 : EPI == 6 ? 1 : 0;        // folded terms of a specialised epilogue
    constexpr bool NOBASE = EPI == 7;
    static_assert(!(PLAIN && MAP), "the specialised epilogues have no material map");
    extern __shared__ __align__(128) unsigned char lsm[];
    // ring of NS plane slots.  Without a material map the planes arrive by cp.async (zero fill outside the sample)
    // three planes ahead of their use; with a map the loader goes through registers (vacuum cells are zeroed).
    constexpr int NS = MAP ? 4 : TMA ? 6 : 5;
    // fp32 tensor copies: a box must start on a 16-byte boundary, so the tile starts FOUR cells left of the block (x0 - 4)
    // and is 72 wide; everywhere else two cells and 68
    constexpr bool WIDE = TMA && sizeof(T) == 4;
    constexpr int PX2 = WIDE ? 72 : k2PX, XO = WIDE ? 4 : 2, TL2 = PX2 * k2HY;
    constexpr int SLOT = (int)(k2_slot_bytes<T, WIDE>() / sizeof(T));             // elements between two plane slots
    static_assert(!(TMA && MAP), "the tensor-copy loader has no vacuum masking");
    T* tiles = reinterpret_cast<T*>(lsm);                                   // [NS][SLOT >= 3 TL2]
    unsigned char* flags = lsm + (size_t)NS * SLOT * sizeof(T);             // [NS][TL2]
    LandauD<T>* smats = reinterpret_cast<LandauD<T>*>(flags + NS * TL2);  // [nmat]
    unsigned char* sact = reinterpret_cast<unsigned char*>(smats + a.nmat);  // [nmat]
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(
        lsm + (((size_t)(sact + a.nmat - lsm) + 7) / 8) * 8);                // [NS] "plane has landed" mbarriers of the tensor-copy loader
    unsigned long long* ebars = bars + NS;                                   // [NS] "every warp is done with the plane" mbarriers
    using P2 = pair_t<T>;

    const int nx = a.n[0], ny = a.n[1], nz = a.n[2];
    const int ntx = (nx + k2TX - 1) / k2TX;
    const int x0 = (blockIdx.x % ntx) * k2TX, y0 = (blockIdx.x / ntx) * kTY;
    const int z0 = a.zbeg + blockIdx.y * a.zchunk, z1 = min(z0 + a.zchunk, a.zend);
    const int b = blockIdx.z;
    const int t = threadIdx.x, tx = t & 31, ty = t >> 5;
    const int64_t nxy = (int64_t)nx * ny, N = nxy * nz;
    const T* Y = static_cast<const T*>(a.Y) + (int64_t)b * 3 * N;
    const DevLandau* mats = a.mats + (int64_t)b * a.nmat;
    for (int m = t; m < a.nmat; m += 256) {
        smats[m] = LandauD<T>(mats[m]);
        sact[m] = mats[m].active != 0;
    }
    const DevMember mem = a.members[b];

    // loader entries: shared offset (-1: none), in-plane global offset of the first cell (-1: outside), pair or single
    int l_so[k2NL], l_go[k2NL];
    bool l_pair[k2NL];
    const T* l_ptr[k2NL];
#pragma unroll
    for (int k = 0; k < k2NL; ++k) {
        const int idx = t + 256 * k;
        l_so[k] = -1;
        l_go[k] = -1;
        l_pair[k] = false;
        l_ptr[k] = Y;
        int comp = 0, yy = 0, col = 0;
        bool have = false;
        if (idx < 3 * k2Pairs) {
            comp = idx / k2Pairs;
            const int rem = idx % k2Pairs;
            yy = rem / (k2TX / 2);
            col = 2 * (rem % (k2TX / 2));            // tile x of the first cell of the pair
            l_pair[k] = true;
            have = true;
        } else if (idx < 3 * (k2Pairs + k2Sing)) {
            const int s2 = idx - 3 * k2Pairs;
            comp = s2 / k2Sing;
            const int rem = s2 % k2Sing;
            yy = rem / 2;
            col = (rem & 1) ? k2TX : -1;
            have = true;
        }
        if (have) {
            int gx = x0 + col, gy = y0 - 1 + yy;
            bool in = true;
            if (gx < 0 || gx >= nx) { if (a.periodic[0]) gx = ((gx % nx) + nx) % nx; else in = false; }
            if (gy < 0 || gy >= ny) { if (a.periodic[1]) gy = ((gy % ny) + ny) % ny; else in = false; }
            l_so[k] = comp * TL2 + yy * PX2 + XO + col;
            l_go[k] = in ? gy * nx + gx : -1;
            if (in) l_ptr[k] = Y + (int64_t)comp * N + l_go[k];
        }
    }
    T pre[k2NL][2];
    bool pok[k2NL][2];
    auto fetch_plane = [&](int z) {
        int zz = z;
        bool zin = true;
        if (zz < 0 || zz >= nz) { if (a.periodic[2]) zz = ((zz % nz) + nz) % nz; else zin = false; }
        const int64_t r0 = (int64_t)zz * nxy;
#pragma unroll
        for (int k = 0; k < k2NL; ++k) {
            const bool ok = zin && l_go[k] >= 0;
            pre[k][0] = pre[k][1] = (T)0;
            pok[k][0] = pok[k][1] = ok;
            if (ok) {
                if (l_pair[k]) {
                    const P2 v = *reinterpret_cast<const P2*>(l_ptr[k] + r0);
                    pre[k][0] = v.a;
                    pre[k][1] = v.b;
                } else {
                    pre[k][0] = l_ptr[k][r0];
                }
                if (MAP) {
                    pok[k][0] = sact[a.map[r0 + l_go[k]]] != 0;
                    if (l_pair[k]) pok[k][1] = sact[a.map[r0 + l_go[k] + 1]] != 0;
                }
            }
        }
    };
    auto slot_of = [&](int z) { return (int)((unsigned)(z - z0 + 1) % NS); };
    auto async_plane = [&](int z) {
        if (z > z1) { asm volatile("cp.async.commit_group;\n" ::); return; }     // not needed: empty group
        int zz = z;
        bool zin = true;
        if (zz < 0 || zz >= nz) { if (a.periodic[2]) zz = ((zz % nz) + nz) % nz; else zin = false; }
        const int64_t r0 = (int64_t)zz * nxy;
        T* tl = tiles + slot_of(z) * SLOT;
#pragma unroll
        for (int k = 0; k < k2NL; ++k) {
            if (l_so[k] < 0) continue;
            const bool ok = zin && l_go[k] >= 0;
            const T* src = ok ? l_ptr[k] + r0 : Y;
            if (l_pair[k]) cp_async_zfill<2 * (int)sizeof(T)>(tl + l_so[k], src, ok ? 2 * (int)sizeof(T) : 0);
            else cp_async_zfill<(int)sizeof(T)>(tl + l_so[k], src, ok ? (int)sizeof(T) : 0);
        }
        asm volatile("cp.async.commit_group;\n" ::);
    };
    auto store_plane = [&](int z) {
        const int slot = slot_of(z);
        T* tl = tiles + slot * SLOT;
        unsigned char* fl = flags + slot * TL2;
#pragma unroll
        for (int k = 0; k < k2NL; ++k) {
            if (l_so[k] < 0) continue;
            if (l_pair[k]) {
                *reinterpret_cast<P2*>(tl + l_so[k]) = P2{pok[k][0] ? pre[k][0] : (T)0, pok[k][1] ? pre[k][1] : (T)0};
                if (MAP && l_so[k] < TL2) { fl[l_so[k]] = pok[k][0]; fl[l_so[k] + 1] = pok[k][1]; }
            } else {
                tl[l_so[k]] = pok[k][0] ? pre[k][0] : (T)0;
                if (MAP && l_so[k] < TL2) fl[l_so[k]] = pok[k][0];
            }
        }
    };
    // tensor-copy loader: plane z of all three components in one copy, completion on the slot's mbarrier
    auto tma_plane = [&](int z) {
        if (z > z1 || t != 0) return;
        const int slot = slot_of(z);
        l_mbar_expect_tx(&bars[slot], (unsigned)(3 * TL2 * sizeof(T)));
        l_tma_load_4d(tiles + slot * SLOT, &tmap, x0 - XO, y0 - 1, z, 3 * b, &bars[slot]);
    };
    auto tma_wait = [&](int z) { l_mbar_wait(&bars[slot_of(z)], (unsigned)(((z - z0 + 1) / NS) & 1)); };
    if (TMA && t == 0) {
        for (int i = 0; i < NS; ++i) { l_mbar_init(&bars[i], 1); l_mbar_init(&ebars[i], 8); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();          // coefficient tables visible (fetch_plane reads sact); mbarriers initialised
    if (MAP) {
        fetch_plane(z0 - 1);
        store_plane(z0 - 1);
        fetch_plane(z0);
        store_plane(z0);
        fetch_plane(z0 + 1);
    } else if (TMA) {
        tma_plane(z0 - 1);
        tma_plane(z0);
        tma_plane(z0 + 1);
        tma_plane(z0 + 2);
        tma_wait(z0 - 1);         // the loop waits for plane z + 1 only: the first two are awaited here
        tma_wait(z0);
    } else {
        async_plane(z0 - 1);
        async_plane(z0);
        async_plane(z0 + 1);
        async_plane(z0 + 2);
    }

    // the tensor-copy loader runs on open grids only: the boundary tests need no periodic flags there
    const bool per0 = !TMA && a.periodic[0], per1 = !TMA && a.periodic[1], per2 = !TMA && a.periodic[2];
    const int x = x0 + 2 * tx, y = y0 + ty;          // cells (x, y) and (x + 1, y)
    const bool inside = x < nx && y < ny;            // nx is even: both cells or none
    const int64_t rxy = (int64_t)y * nx + x;
    const int c0 = (ty + 1) * PX2 + XO + 2 * tx;
    const T gxfA = (T)((x > 0 || per0) + 1), gxfB = (T)(1 + (x + 2 < nx || per0));
    const T gyf = (T)((y > 0 || per1) + (y < ny - 1 || per1));
    const T G11 = (T)mem.G11, Gt = (T)mem.Gt, Gm = (T)mem.Gm, L = (T)mem.L;
    const T ix = (T)a.id2[0], iy = (T)a.id2[1], iz = (T)a.id2[2];
    const T qxy = Gm * (T)a.i4[0], qxz = Gm * (T)a.i4[1], qyz = Gm * (T)a.i4[2];
    const T cy = (T)a.cy, ca = (T)a.ca;
    const double wv = mem.wave ? sin(mem.womega * a.t + mem.wphase) : 0.0;      // E_ext sampled at the stage time
    const T ex0 = (T)(mem.Eext[0] + mem.wamp[0] * wv), ex1 = (T)(mem.Eext[1] + mem.wamp[1] * wv),
            ex2 = (T)(mem.Eext[2] + mem.wamp[2] * wv);
    const uint32_t terms = PLAIN ? 15u : a.terms;
    const T* Ee = PLAIN || ((terms & 4u) && a.Eelec) ? static_cast<const T*>(a.Eelec) + (int64_t)b * 3 * N : nullptr;
    const T* base = BASEY ? Y : NOBASE ? nullptr : (PLAIN || a.baseY) ? static_cast<const T*>(a.baseY) + (int64_t)b * 3 * N : nullptr;
    const bool base_is_Y = BASEY || (!PLAIN && a.baseY == a.Y);
    T* Yout = static_cast<T*>(a.Yout) + (int64_t)b * 3 * N;
    const T* ai = (ACC || (!PLAIN && a.accOut)) ? static_cast<const T*>(a.accIn) + (int64_t)b * 3 * N : nullptr;
    T* ao = (ACC || (!PLAIN && a.accOut)) ? static_cast<T*>(a.accOut) + (int64_t)b * 3 * N : nullptr;
    const int nlin = PLAIN ? NLIN : a.nlin;
    const LandauD<T> lc0 = smats[0];
    auto ldp = [](const T* q) { return *reinterpret_cast<const P2*>(q); };

    // PLAIN: the thread's own cell pair of planes z-1 and z rides in registers from plane to plane (6 of the 45 loads)
    P2 cz[3] = {{0, 0}, {0, 0}, {0, 0}}, cc[3] = {{0, 0}, {0, 0}, {0, 0}};
    if (PLAIN && !TMA) {
        asm volatile("cp.async.wait_group 2;\n" ::);            // planes z0 - 1 and z0 of the four requested have landed
        __syncthreads();
    }
    if (PLAIN && inside) {
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            cz[i] = ldp(tiles + i * TL2 + c0);               // plane z0 - 1 sits in slot 0,
            cc[i] = ldp(tiles + SLOT + i * TL2 + c0);        // plane z0 in slot 1
        }
    }
    // slots of planes z-1, z, z+1 and the phase bits of the slots' mbarriers, carried from plane to plane (no division per plane)
    int sm1 = 0, s00 = 1, sp1 = 2;
    unsigned phases = 3u;                            // slots 0 and 1 were awaited once in the prologue
    unsigned ephases = 0u;                           // thread 0: phase bits of the release mbarriers
    int64_t r = (int64_t)z0 * nxy + rxy;             // cell pair (x, y, z) of this thread
    for (int z = z0; z < z1; ++z, r += nxy, sm1 = s00, s00 = sp1, sp1 = (sp1 + 1 == NS ? 0 : sp1 + 1)) {
        // E_elec of this plane: requested before the wait for the next halo plane, consumed after the stencil
        P2 ec[3] = {{0, 0}, {0, 0}, {0, 0}};
        if (Ee && inside) {
#pragma unroll
            for (int i = 0; i < 3; ++i) ec[i] = ldp(Ee + i * N + r);
        }
        if (MAP) {
            store_plane(z + 1);
            __syncthreads();
            if (z + 1 < z1) fetch_plane(z + 2);      // in flight while plane z is computed
        } else if (TMA) {
            // no block barrier: a warp releases plane z-2 (last read in its iteration z-1) on the slot's second mbarrier,
            // and thread 0 refills the slot of plane z-3 once all eight warps have released it
            if (z > z0) {
                __syncwarp();
                if ((t & 31) == 0) l_mbar_arrive(&ebars[sm1 == 0 ? NS - 1 : sm1 - 1]);
            }
            l_mbar_wait(&bars[sp1], (phases >> sp1) & 1u);   // planes <= z+1 have landed
            phases ^= 1u << sp1;
            if (t == 0 && z + 3 <= z1) {                     // plane z+3 into the slot of plane z-3
                const int s3 = sp1 + 2 >= NS ? sp1 + 2 - NS : sp1 + 2;
                if (z - z0 >= 2) {                           // (the first NS planes find their slots fresh)
                    l_mbar_wait(&ebars[s3], (ephases >> s3) & 1u);
                    ephases ^= 1u << s3;
                }
                l_mbar_expect_tx(&bars[s3], (unsigned)(3 * TL2 * sizeof(T)));
                l_tma_load_4d(tiles + s3 * SLOT, &tmap, x0 - XO, y0 - 1, z + 3, 3 * b, &bars[s3]);
            }
        } else {
            asm volatile("cp.async.wait_group 1;\n" ::);     // planes <= z+1 have landed
            __syncthreads();
            async_plane(z + 3);                              // into the slot of plane z-2 (commits a group)
        }
        if (!inside) continue;
        const T* m0 = tiles + sm1 * SLOT;           // plane z-1
        const T* c = tiles + s00 * SLOT;            // plane z
        const T* p1 = tiles + sp1 * SLOT;           // plane z+1
        const unsigned char* fm = flags + sm1 * TL2;
        const unsigned char* fc = flags + s00 * TL2;
        const unsigned char* fp = flags + sp1 * TL2;
        // without a map every cell is material 0 (a vacuum material 0 pins the whole member: VAC)
        const bool act0 = !VAC || lc0.active != 0;
        const bool actA = MAP ? fc[c0] != 0 : act0, actB = MAP ? fc[c0 + 1] != 0 : act0;
        T EA[3] = {0, 0, 0}, EB[3] = {0, 0, 0};
        P2 pc[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) pc[i] = PLAIN ? cc[i] : ldp(c + i * TL2 + c0);
        if (terms & 1u) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const LandauD<T> lc = MAP ? smats[a.map[r + h]] : lc0;
                const T px = h ? pc[0].b : pc[0].a, py = h ? pc[1].b : pc[1].a, pz = h ? pc[2].b : pc[2].a;
                const T A = px * px, B = py * py, C = pz * pz;
                const T A2 = A * A, B2 = B * B, C2 = C * C;
                T A3 = 0, B3 = 0, C3 = 0;
                if (lc.o8) { A3 = A2 * A; B3 = B2 * B; C3 = C2 * C; }
                T* E = h ? EB : EA;
                E[0] -= px * lc.dfd(lc.k1x, A, A2, B + C, B2 + C2, B * C, B3 + C3);
                E[1] -= py * lc.dfd(lc.k1y, B, B2, C + A, C2 + A2, C * A, C3 + A3);
                E[2] -= pz * lc.dfd(lc.k1z, C, C2, A + B, A2 + B2, A * B, A3 + B3);
            }
        }
        if (terms & 2u) {
            // number of existing neighbours per axis (a missing neighbour holds 0 in the tile)
            const T nzg = (T)((z > 0 || per2) + (z < nz - 1 || per2));
            const T nxA = MAP ? (T)(fc[c0 - 1] + fc[c0 + 1]) : gxfA, nxB = MAP ? (T)(fc[c0] + fc[c0 + 2]) : gxfB;
            const T nyA = MAP ? (T)(fc[c0 - PX2] + fc[c0 + PX2]) : gyf;
            const T nyB = MAP ? (T)(fc[c0 + 1 - PX2] + fc[c0 + 1 + PX2]) : gyf;
            const T nzA = MAP ? (T)(fm[c0] + fp[c0]) : nzg, nzB = MAP ? (T)(fm[c0 + 1] + fp[c0 + 1]) : nzg;
            // taps shared by the bond sums and the mixed term: rows y-1 / y+1 of plane z, planes z-1 / z+1 at row y
            P2 dn[3], up[3], zm[3], zp[3];
            T lf[3], rt[3];
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                const T* ci = c + i * TL2 + c0;
                dn[i] = ldp(ci - PX2);
                up[i] = ldp(ci + PX2);
                zm[i] = PLAIN ? cz[i] : ldp(m0 + i * TL2 + c0);
                zp[i] = ldp(p1 + i * TL2 + c0);
                if (PLAIN) { cz[i] = pc[i]; cc[i] = zp[i]; }
                lf[i] = ci[-1];
                rt[i] = ci[2];
                const T gx_ = (i == 0 ? G11 : Gt) * ix, gy_ = (i == 1 ? G11 : Gt) * iy, gz_ = (i == 2 ? G11 : Gt) * iz;
                EA[i] += gx_ * (lf[i] + pc[i].b - nxA * pc[i].a) + gy_ * (dn[i].a + up[i].a - nyA * pc[i].a) +
                         gz_ * (zm[i].a + zp[i].a - nzA * pc[i].a);
                EB[i] += gx_ * (pc[i].a + rt[i] - nxB * pc[i].b) + gy_ * (dn[i].b + up[i].b - nyB * pc[i].b) +
                         gz_ * (zm[i].b + zp[i].b - nzB * pc[i].b);
            }
            if (MIXED) {
                // Gm sum_{j != i} [P_j(+i+j) - P_j(+i-j) - P_j(-i+j) + P_j(-i-j)] / (4 D_i D_j); columns -1 .. +2 around cell A
                const T* cxp = c + c0;
                const T* cyp = c + TL2 + c0;
                const T* czm = m0 + 2 * TL2 + c0;
                const T* czp = p1 + 2 * TL2 + c0;
                // xy: Py and Px on rows y+-1
                const T yul = cyp[PX2 - 1], yur = cyp[PX2 + 2], ydl = cyp[-PX2 - 1], ydr = cyp[-PX2 + 2];
                const T xul = cxp[PX2 - 1], xur = cxp[PX2 + 2], xdl = cxp[-PX2 - 1], xdr = cxp[-PX2 + 2];
                EA[0] += qxy * (up[1].b - dn[1].b - yul + ydl);
                EB[0] += qxy * (yur - ydr - up[1].a + dn[1].a);
                EA[1] += qxy * (up[0].b - dn[0].b - xul + xdl);
                EB[1] += qxy * (xur - xdr - up[0].a + dn[0].a);
                // xz: Pz and Px on planes z+-1 at row y
                const T zpl = czp[-1], zpr = czp[2], zml = czm[-1], zmr = czm[2];
                const T* cxm = m0 + c0;
                const T* cxq = p1 + c0;
                const T xpl = cxq[-1], xpr = cxq[2], xml = cxm[-1], xmr = cxm[2];
                EA[0] += qxz * (zp[2].b - zm[2].b - zpl + zml);
                EB[0] += qxz * (zpr - zmr - zp[2].a + zm[2].a);
                EA[2] += qxz * (zp[0].b - zm[0].b - xpl + xml);
                EB[2] += qxz * (xpr - xmr - zp[0].a + zm[0].a);
                // yz: Pz and Py on planes z+-1 at rows y+-1
                const P2 zpu = ldp(czp + PX2), zpd = ldp(czp - PX2), zmu = ldp(czm + PX2), zmd = ldp(czm - PX2);
                const T* cym = m0 + TL2 + c0;
                const T* cyq = p1 + TL2 + c0;
                const P2 ypu = ldp(cyq + PX2), ypd = ldp(cyq - PX2), ymu = ldp(cym + PX2), ymd = ldp(cym - PX2);
                EA[1] += qyz * (zpu.a - zmu.a - zpd.a + zmd.a);
                EB[1] += qyz * (zpu.b - zmu.b - zpd.b + zmd.b);
                EA[2] += qyz * (ypu.a - ypd.a - ymu.a + ymd.a);
                EB[2] += qyz * (ypu.b - ypd.b - ymu.b + ymd.b);
            }
        }
        T kA[3] = {0, 0, 0}, kB[3] = {0, 0, 0};
        if (Ee) {
#pragma unroll
            for (int i = 0; i < 3; ++i) { EA[i] += ec[i].a; EB[i] += ec[i].b; }
        }
        if (terms & 8u) {
            EA[0] += ex0; EA[1] += ex1; EA[2] += ex2;
            EB[0] += ex0; EB[1] += ex1; EB[2] += ex2;
        }
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            if (actA) kA[i] = L * EA[i];
            if (actB) kB[i] = L * EB[i];
        }
        if (KOUT || (!PLAIN && a.kOut)) {
            T* ko = static_cast<T*>(a.kOut) + (int64_t)b * 3 * N;
#pragma unroll
            for (int i = 0; i < 3; ++i) *reinterpret_cast<P2*>(ko + i * N + r) = P2{kA[i], kB[i]};
        }
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            P2 bv = {0, 0};
            if (!NOBASE && (PLAIN || base)) {
                // Euler: the stage base is the state itself, already in the tile (vacuum cells hold their raw value in memory)
                if (base_is_Y && actA && actB) bv = pc[i];
                else bv = ldp(base + i * N + r);
            }
            for (int j = 0; j < nlin; ++j) {
                const P2 lv = ldp(static_cast<const T*>(a.lk[j]) + (int64_t)b * 3 * N + i * N + r);
                const T cj = (T)a.lc[j];
                bv = P2{bv.a + cj * lv.a, bv.b + cj * lv.b};
            }
            *reinterpret_cast<P2*>(Yout + i * N + r) = P2{bv.a + cy * kA[i], bv.b + cy * kB[i]};
            if (ACC || ao) {
                const P2 av = ldp(ai + i * N + r);
                *reinterpret_cast<P2*>(ao + i * N + r) = P2{av.a + ca * kA[i], av.b + ca * kB[i]};
            }
        }
    }

}

// Tensor map of a state array [B * 3][nz][ny][nx] with the 68 x 10 x 1 x 3 box of k_local2's plane slots.  The encoder is
// a driver entry point fetched at run time (no link against libcuda).  Returns false when the geometry does not meet the
// copy engine's rules (row pitch a multiple of 16 bytes) or the entry point is missing: the caller uses cp.async then.
template <typename T> static bool make_state_map(const LocalArgs& a, CUtensorMap* out)
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
    // the box starts two cells left of the tile in fp64 (x0 - 2: 16 bytes) and four in fp32 (an 8-byte-aligned start raised
    // an illegal-instruction fault in the copy engine on B200), where it is 72 cells wide
    const cuuint32_t bx = sizeof(T) == 8 ? k2PX : 72;
    const cuuint64_t nx = a.n[0], ny = a.n[1], nz = a.n[2];
    if ((nx * sizeof(T)) % 16 || nx < (cuuint64_t)bx || ny < (cuuint64_t)k2HY) return false;
    if (reinterpret_cast<uintptr_t>(a.Y) % 16) return false;
    const cuuint64_t dims[4] = {nx, ny, nz, (cuuint64_t)3 * a.batch};
    const cuuint64_t strides[3] = {nx * sizeof(T), nx * ny * sizeof(T), nx * ny * nz * sizeof(T)};
    const cuuint32_t box[4] = {bx, (cuuint32_t)k2HY, 1, 3};
    const cuuint32_t es[4] = {1, 1, 1, 1};
    const CUresult r = enc(out, sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4,
                           const_cast<void*>(a.Y), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

template <typename T> cudaError_t launch_local(const LocalArgs& a0, cudaStream_t st)
{
    LocalArgs a = a0;
    for (int i = 0; i < 3; ++i) a.id2[i] = 1.0 / (a.d[i] * a.d[i]);
    a.i4[0] = 0.25 / (a.d[0] * a.d[1]);
    a.i4[1] = 0.25 / (a.d[0] * a.d[2]);
    a.i4[2] = 0.25 / (a.d[1] * a.d[2]);
    const bool two = a.n[0] >= k2TX;      // two cells per thread on rows of at least 64 cells
    const int ntx = two ? (a.n[0] + k2TX - 1) / k2TX : (a.n[0] + kTX - 1) / kTX, nty = (a.n[1] + kTY - 1) / kTY;
    // z chunk: as long as possible (halo planes are re-read per chunk) while the grid still fills the machine
    if (a.zend <= 0) { a.zbeg = 0; a.zend = a.n[2]; }
    // a slab buffer holds plane z of a component at plane z - e_z0 of the component's region: fold that into the pointer
    if (a.Eelec && a.e_z0) a.Eelec = static_cast<const T*>(a.Eelec) - (int64_t)a.e_z0 * a.n[0] * a.n[1];
    const int nzl = a.zend - a.zbeg;      // planes of this launch
    int zc = nzl;
    while (zc > 8 && (int64_t)ntx * nty * ((nzl + zc - 1) / zc) * a.batch < 12 * 148) zc = (zc + 1) / 2;
    a.zchunk = zc;
    dim3 grid(ntx * nty, (nzl + zc - 1) / zc, a.batch);
    // halo planes by tensor copy (zero fill outside the sample) when there is neither a material map nor a periodic axis
    CUtensorMap tmap;
    memset(&tmap, 0, sizeof(tmap));
    const bool tma = two && !a.map && !(a.periodic[0] | a.periodic[1] | a.periodic[2]) && make_state_map<T>(a, &tmap);
    const int ns = a.map ? 4 : tma ? 6 : 5;         // ring slots of k_local2
    const bool wide = tma && sizeof(T) == 4;      // fp32 tensor copies: 72-wide tiles (see k_local2)
    const size_t slot_bytes = wide ? k2_slot_bytes<T, true>() : k2_slot_bytes<T>();
    const size_t smem = two ? (size_t)ns * slot_bytes + ns * (wide ? 72 * k2HY : k2Tile) + (size_t)a.nmat * (sizeof(LandauD<T>) + 1) + 8 + 2 * ns * 8
                            : (size_t)4 * 3 * kTile * sizeof(T) + 4 * kTile + 8 + (size_t)a.nmat * (sizeof(LandauD<T>) + 1);
    static PerDevice<int> cache;
    int& configured = cache.here();
    if (!configured) {
        const int lim = 96 * 1024;      // 255 materials need 61 KB
        cudaError_t e = cudaFuncSetAttribute(k_local<T, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_local<T, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_local<T, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_local<T, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim);
        const int lim2 = 128 * 1024;
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_local2<T, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim2);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_local2<T, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim2);
        auto attr = [&](auto m, auto tm, auto ep) {
            if (e == cudaSuccess)
                e = cudaFuncSetAttribute(k_local2<T, false, decltype(m)::value, decltype(tm)::value, decltype(ep)::value>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, lim2);
        };
        auto a2 = [&](auto m, auto tm) {
            attr(m, tm, std::integral_constant<int, 0>{});
            attr(m, tm, std::integral_constant<int, 1>{});
            attr(m, tm, std::integral_constant<int, 2>{});
            attr(m, tm, std::integral_constant<int, 3>{});
            attr(m, tm, std::integral_constant<int, 4>{});
            attr(m, tm, std::integral_constant<int, 5>{});
            attr(m, tm, std::integral_constant<int, 6>{});
            attr(m, tm, std::integral_constant<int, 7>{});
        };
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_local2<T, false, true, true, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim2);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_local2<T, false, false, true, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim2);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_local2<T, false, true, false, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim2);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_local2<T, false, false, false, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim2);
        a2(std::true_type{}, std::true_type{});
        a2(std::true_type{}, std::false_type{});
        a2(std::false_type{}, std::true_type{});
        a2(std::false_type{}, std::false_type{});
        if (e != cudaSuccess) return e;
        configured = 1;
    }
    if (two) {
        if (a.map) {
            if (a.mixed) k_local2<T, true, true><<<grid, 256, smem, st>>>(a, tmap);
            else k_local2<T, true, false><<<grid, 256, smem, st>>>(a, tmap);
        } else {
            // a stage of Euler / Heun / RK4 with all four terms: one of the specialised epilogues (see k_local2)
            const bool full = a.terms == 15u && a.Eelec && a.baseY;
            int epi = 0;
            if (a.vac0) {                  // some member is all vacuum: general epilogue with the activity check
                if (tma) {
                    if (a.mixed) k_local2<T, false, true, true, 0, true><<<grid, 256, smem, st>>>(a, tmap);
                    else k_local2<T, false, false, true, 0, true><<<grid, 256, smem, st>>>(a, tmap);
                } else {
                    if (a.mixed) k_local2<T, false, true, false, 0, true><<<grid, 256, smem, st>>>(a, tmap);
                    else k_local2<T, false, false, false, 0, true><<<grid, 256, smem, st>>>(a, tmap);
                }
                return cudaGetLastError();
            }
            if (a.terms == 15u && a.Eelec && !a.baseY && !a.kOut && a.nlin == 0 && !a.accOut) epi = 7;
            if (full && !a.kOut && a.nlin == 0) epi = a.baseY == a.Y ? (a.accOut ? 2 : 1) : (a.accOut ? 4 : 3);
            else if (full && a.kOut && a.nlin == 2 && a.baseY == a.Y && !a.accOut) epi = 5;
            else if (full && !a.kOut && a.nlin == 1 && a.baseY != a.Y && !a.accOut) epi = 6;
            auto go = [&](auto m, auto tm, auto ep) {
                k_local2<T, false, decltype(m)::value, decltype(tm)::value, decltype(ep)::value><<<grid, 256, smem, st>>>(a, tmap);
            };
            auto d2 = [&](auto m, auto tm) {
                switch (epi) {
                    case 1: go(m, tm, std::integral_constant<int, 1>{}); break;
                    case 2: go(m, tm, std::integral_constant<int, 2>{}); break;
                    case 3: go(m, tm, std::integral_constant<int, 3>{}); break;
                    case 4: go(m, tm, std::integral_constant<int, 4>{}); break;
                    case 5: go(m, tm, std::integral_constant<int, 5>{}); break;
                    case 6: go(m, tm, std::integral_constant<int, 6>{}); break;
                    case 7: go(m, tm, std::integral_constant<int, 7>{}); break;
                    default: go(m, tm, std::integral_constant<int, 0>{}); break;
                }
            };
            auto d1 = [&](auto m) { if (tma) d2(m, std::true_type{}); else d2(m, std::false_type{}); };
            if (a.mixed) d1(std::true_type{}); else d1(std::false_type{});
        }
        return cudaGetLastError();
    }
    if (a.map) {
        if (a.mixed) k_local<T, true, true><<<grid, 256, smem, st>>>(a);
        else k_local<T, true, false><<<grid, 256, smem, st>>>(a);
    } else {
        if (a.mixed) k_local<T, false, true><<<grid, 256, smem, st>>>(a);
        else k_local<T, false, false><<<grid, 256, smem, st>>>(a);
    }
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// a6: energies and means (Eq. 2, 66 Eq. 5, 80 Eq. 7, 121).  fp64 accumulation in both modes;
// warp-shuffle reduction, one partial row per block, a second tiny kernel sums the rows (deterministic).
//   F_Land = V sum f_Land;  F_Grad = V sum_r { sum_i sum_a c_ia/2 [(P_i(r+e_a)-P_i(r))/D_a]^2 (bond exists)
//            + Gm sum_{i<j} D_iP_i D_jP_j };  F_Elec = -V/2 sum E_Elec.P;  F_Ext = -V sum E_Ext.P
// ------------------------------------------------------------------------------------------------
constexpr int kEn = 8;   // F_Land, F_Grad, F_Elec, F_Ext, sumPx, sumPy, sumPz, n_active

template <typename T, bool MAP>
__global__ void __launch_bounds__(256) k_energy(EnergyArgs a)
{
    const int nx = a.n[0], ny = a.n[1], nz = a.n[2];
    const int64_t N = (int64_t)nx * ny * nz;
    const int b = blockIdx.y;
    const T* P = static_cast<const T*>(a.P) + (int64_t)b * 3 * N;
    const DevLandau* mats = a.mats + (int64_t)b * a.nmat;
    const DevMember mem = a.members[b];
    Grid<T, MAP> g{{P, P + N, P + 2 * N}, a.map, mats, nx, ny, nz};
    double acc[kEn] = {0, 0, 0, 0, 0, 0, 0, 0};
    const double Gt = mem.Gt, G11 = mem.G11, Gm = mem.Gm;
    const double wv = mem.wave ? sin(mem.womega * a.t + mem.wphase) : 0.0;
    const double eex[3] = {mem.Eext[0] + mem.wamp[0] * wv, mem.Eext[1] + mem.wamp[1] * wv, mem.Eext[2] + mem.wamp[2] * wv};
    for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r < N; r += (int64_t)gridDim.x * blockDim.x) {
        const int x = (int)(r % nx), y = (int)((r / nx) % ny), z = (int)(r / ((int64_t)nx * ny));
        const int c0[3] = {x, y, z};
        const int mat = MAP ? a.map[r] : 0;
        const bool act = mats[mat].active != 0;
        const double p0[3] = {act ? (double)P[r] : 0.0, act ? (double)P[N + r] : 0.0, act ? (double)P[2 * N + r] : 0.0};
        if (act) {
            if (a.terms & 1u) {
                const LandauT<double> L(mats[mat]);
                acc[0] += L.f(p0[0] * p0[0], p0[1] * p0[1], p0[2] * p0[2]);
            }
            if ((a.terms & 4u) && a.Eelec) {
                const T* Ee = static_cast<const T*>(a.Eelec) + (int64_t)b * 3 * N;
                acc[2] -= 0.5 * ((double)Ee[r] * p0[0] + (double)Ee[N + r] * p0[1] + (double)Ee[2 * N + r] * p0[2]);
            }
            if (a.terms & 8u) acc[3] -= eex[0] * p0[0] + eex[1] * p0[1] + eex[2] * p0[2];
            acc[4] += p0[0]; acc[5] += p0[1]; acc[6] += p0[2]; acc[7] += 1.0;
        }
        if (a.terms & 2u) {
            double D[3];
            for (int ax = 0; ax < 3; ++ax) {
                int qp[3] = {x, y, z}, qm[3] = {x, y, z};
                qp[ax] = nb(c0[ax], +1, a.n[ax], a.periodic[ax]);
                qm[ax] = nb(c0[ax], -1, a.n[ax], a.periodic[ax]);
                bool okp;
                const double upx = (double)g.val(0, qp[0], qp[1], qp[2], okp);
                if (act && okp) {      // forward bond, counted once
                    const int64_t rq = ((int64_t)qp[2] * ny + qp[1]) * nx + qp[0];
                    const double u[3] = {upx, (double)P[N + rq], (double)P[2 * N + rq]};
                    for (int i = 0; i < 3; ++i) {
                        const double q = (u[i] - p0[i]) / a.d[ax];
                        acc[1] += 0.5 * (i == ax ? G11 : Gt) * q * q;
                    }
                }
                const double up = (double)g.val(ax, qp[0], qp[1], qp[2]);
                const double dn = (double)g.val(ax, qm[0], qm[1], qm[2]);
                D[ax] = (up - dn) / (2.0 * a.d[ax]);
            }
            acc[1] += Gm * (D[0] * D[1] + D[1] * D[2] + D[2] * D[0]);
        }
    }
    __shared__ double red[8][kEn];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < kEn; ++k) {
        double v = acc[k];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) red[warp][k] = v;
    }
    __syncthreads();
    if (threadIdx.x < kEn) {
        double v = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) v += red[w][threadIdx.x];
        a.partials[((int64_t)b * gridDim.x + blockIdx.x) * kEn + threadIdx.x] = v;
    }
}

// out[b] = { F_Land, F_Grad, F_Elec, F_Ext, F_tot, <Px>, <Py>, <Pz> }
__global__ void k_energy_final(const double* __restrict__ partials, double* __restrict__ out, int nblk, double V)
{
    const int b = blockIdx.x;
    __shared__ double s[kEn];
    if (threadIdx.x < kEn) {
        double v = 0.0;
        for (int i = 0; i < nblk; ++i) v += partials[((int64_t)b * nblk + i) * kEn + threadIdx.x];
        s[threadIdx.x] = v;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const double na = s[7] > 0.5 ? s[7] : 1.0;
        double* o = out + b * 8;
        o[0] = V * s[0]; o[1] = V * s[1]; o[2] = V * s[2]; o[3] = V * s[3];
        o[4] = o[0] + o[1] + o[2] + o[3];
        o[5] = s[4] / na; o[6] = s[5] / na; o[7] = s[6] / na;
    }
}

template <typename T> cudaError_t launch_energy(const EnergyArgs& a, cudaStream_t st)
{
    dim3 grid(a.nblk, a.batch);
    if (a.map) k_energy<T, true><<<grid, 256, 0, st>>>(a);
    else k_energy<T, false><<<grid, 256, 0, st>>>(a);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    k_energy_final<<<a.batch, 32, 0, st>>>(a.partials, a.out, a.nblk, a.d[0] * a.d[1] * a.d[2]);
    return cudaGetLastError();
}

template cudaError_t launch_local<double>(const LocalArgs&, cudaStream_t);
template cudaError_t launch_local<float>(const LocalArgs&, cudaStream_t);
template cudaError_t launch_energy<double>(const EnergyArgs&, cudaStream_t);
template cudaError_t launch_energy<float>(const EnergyArgs&, cudaStream_t);

}  // namespace fe
