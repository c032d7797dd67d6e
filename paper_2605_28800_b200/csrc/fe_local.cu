// fe_local.cu -- a4/a5: fused local step, and a6: energy reduction.
//   k = L * active * (E_Land + E_Grad + E_Elec + E_Ext)                      PAPER.md:33 (Eq. 1)
//   E_Land = -d f_Land/dP, f_Land of Eq. 3 with per-axis a1 and four 8th-order slots
//   E_Grad = exact gradient of the discrete Eq. 4 energy (reading A2):
//            sum_a c_ia [P_i(r+e_a) - 2 P_i(r) + P_i(r-e_a)] / D_a^2   (bond missing -> that difference is 0)
//          + Gm sum_{j != i} [D_j P_j (r+e_i) - D_j P_j (r-e_i)] / (2 D_i), D_j = centred difference with
//            zero outside the sample / in vacuum cells, c_ia = G11 (a == i) or G44 + G44', Gm = G12 + G44 - G44'
//   then the integrator stage:  Yout = baseY + cy * k,  accOut = accIn + ca * k
#include "fe_internal.h"

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
        if (MAP) {
            if (!mats[map[r]].active) { ok = false; return (T)0; }
        }
        ok = true;
        return p[c][r];
    }
    __device__ __forceinline__ T val(int c, int x, int y, int z) const
    {
        bool ok;
        return val(c, x, y, z, ok);
    }
};

template <typename T, bool MAP, bool MIXED>
__global__ void __launch_bounds__(256) k_local(LocalArgs a)
{
    const int nx = a.n[0], ny = a.n[1], nz = a.n[2];
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int yz = blockIdx.y;
    const int y = yz % ny, z = yz / ny;
    const int b = blockIdx.z;
    if (x >= nx) return;
    const int64_t N = (int64_t)nx * ny * nz;
    const int64_t r = ((int64_t)z * ny + y) * nx + x;
    const T* Y = static_cast<const T*>(a.Y) + (int64_t)b * 3 * N;
    const DevLandau* mats = a.mats + (int64_t)b * a.nmat;
    const DevMember mem = a.members[b];
    const int mat = MAP ? a.map[r] : 0;
    const bool act = mats[mat].active != 0;

    T k[3] = {0, 0, 0};
    if (act) {
        const T p0[3] = {Y[r], Y[N + r], Y[2 * N + r]};
        T E[3] = {0, 0, 0};
        if (a.terms & 1u) {
            const LandauT<T> L(mats[mat]);
            const T A = p0[0] * p0[0], B = p0[1] * p0[1], C = p0[2] * p0[2];
            E[0] -= p0[0] * L.dfd(L.a1x, A, B, C);
            E[1] -= p0[1] * L.dfd(L.a1y, B, C, A);
            E[2] -= p0[2] * L.dfd(L.a1z, C, A, B);
        }
        if (a.terms & 2u) {
            Grid<T, MAP> g{{Y, Y + N, Y + 2 * N}, a.map, mats, nx, ny, nz};
            const int c0[3] = {x, y, z};
            const T G11 = (T)mem.G11, Gt = (T)mem.Gt;
            const T id2[3] = {(T)(1.0 / (a.d[0] * a.d[0])), (T)(1.0 / (a.d[1] * a.d[1])), (T)(1.0 / (a.d[2] * a.d[2]))};
#pragma unroll
            for (int ax = 0; ax < 3; ++ax) {
#pragma unroll
                for (int s = -1; s <= 1; s += 2) {
                    int q[3] = {c0[0], c0[1], c0[2]};
                    q[ax] = nb(c0[ax], s, a.n[ax], a.periodic[ax]);
                    bool ok;
                    const T vx = g.val(0, q[0], q[1], q[2], ok);
                    if (ok) {
                        const T vy = g.p[1][((int64_t)q[2] * ny + q[1]) * nx + q[0]];
                        const T vz = g.p[2][((int64_t)q[2] * ny + q[1]) * nx + q[0]];
                        E[0] += (ax == 0 ? G11 : Gt) * id2[ax] * (vx - p0[0]);
                        E[1] += (ax == 1 ? G11 : Gt) * id2[ax] * (vy - p0[1]);
                        E[2] += (ax == 2 ? G11 : Gt) * id2[ax] * (vz - p0[2]);
                    }
                }
            }
            if (MIXED) {
                const T Gm = (T)mem.Gm;
                if (Gm != (T)0) {
#pragma unroll
                    for (int i = 0; i < 3; ++i) {
                        T acc = 0;
#pragma unroll
                        for (int j = 0; j < 3; ++j) {
                            if (j == i) continue;
                            T t = 0;
#pragma unroll
                            for (int si = -1; si <= 1; si += 2) {
                                const int ci = nb(c0[i], si, a.n[i], a.periodic[i]);
                                if (ci < 0) continue;      // intermediate cell must be inside the grid
                                int qp[3] = {c0[0], c0[1], c0[2]}, qm[3] = {c0[0], c0[1], c0[2]};
                                qp[i] = ci; qm[i] = ci;
                                qp[j] = nb(c0[j], +1, a.n[j], a.periodic[j]);
                                qm[j] = nb(c0[j], -1, a.n[j], a.periodic[j]);
                                const T up = g.val(j, qp[0], qp[1], qp[2]);
                                const T dn = g.val(j, qm[0], qm[1], qm[2]);
                                t += (T)si * (up - dn);
                            }
                            acc += t * (T)(0.25 / (a.d[i] * a.d[j]));
                        }
                        E[i] += Gm * acc;
                    }
                }
            }
        }
        if ((a.terms & 4u) && a.Eelec) {
            const T* Ee = static_cast<const T*>(a.Eelec) + (int64_t)b * 3 * N;
            E[0] += Ee[r]; E[1] += Ee[N + r]; E[2] += Ee[2 * N + r];
        }
        if (a.terms & 8u) {
            E[0] += (T)mem.Eext[0]; E[1] += (T)mem.Eext[1]; E[2] += (T)mem.Eext[2];
        }
        const T L = (T)mem.L;
        k[0] = L * E[0]; k[1] = L * E[1]; k[2] = L * E[2];
    }
    T* Yout = static_cast<T*>(a.Yout) + (int64_t)b * 3 * N;
    const T* base = a.baseY ? static_cast<const T*>(a.baseY) + (int64_t)b * 3 * N : nullptr;
    const T cy = (T)a.cy;
#pragma unroll
    for (int c = 0; c < 3; ++c) Yout[c * N + r] = (base ? base[c * N + r] : (T)0) + cy * k[c];
    if (a.accOut) {
        const T* ai = static_cast<const T*>(a.accIn) + (int64_t)b * 3 * N;
        T* ao = static_cast<T*>(a.accOut) + (int64_t)b * 3 * N;
        const T ca = (T)a.ca;
#pragma unroll
        for (int c = 0; c < 3; ++c) ao[c * N + r] = ai[c * N + r] + ca * k[c];
    }
}

template <typename T> cudaError_t launch_local(const LocalArgs& a, cudaStream_t st)
{
    const int bx = a.n[0] >= 256 ? 256 : (a.n[0] >= 128 ? 128 : (a.n[0] >= 64 ? 64 : 32));
    dim3 grid((a.n[0] + bx - 1) / bx, a.n[1] * a.n[2], a.batch);
    if (a.map) {
        if (a.mixed) k_local<T, true, true><<<grid, bx, 0, st>>>(a);
        else k_local<T, true, false><<<grid, bx, 0, st>>>(a);
    } else {
        if (a.mixed) k_local<T, false, true><<<grid, bx, 0, st>>>(a);
        else k_local<T, false, false><<<grid, bx, 0, st>>>(a);
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
            if (a.terms & 8u) acc[3] -= mem.Eext[0] * p0[0] + mem.Eext[1] * p0[1] + mem.Eext[2] * p0[2];
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
