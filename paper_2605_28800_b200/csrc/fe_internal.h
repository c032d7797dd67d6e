// fe_internal.h -- host-side declarations shared by the translation units of libfe_b200.
// Not part of the ABI (include/fe.h is).  No code here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

namespace fe {

constexpr int kTwiddleN = 2048;      // twiddle table w[k] = exp(-2 pi i k / 2048); covers every axis length
constexpr int kMaxStages = 6;
constexpr int kThreads = 256;

// One-time kernel set-up (dynamic shared-memory limit, persistent grid size) is a property of the DEVICE, not of the
// process: the launchers cache it per device in a zero-initialised static PerDevice<int>.  Concurrent first calls
// repeat the same idempotent set-up and store the same value.
constexpr int kMaxDevices = 64;
template <typename V> struct PerDevice {
    V v[kMaxDevices];
    V& here()
    {
        int d = 0;
        if (cudaGetDevice(&d) != cudaSuccess || d < 0 || d >= kMaxDevices) d = 0;
        return v[d];
    }
};

// Radix plan of one in-place power-of-two FFT of length M (complex points).
// Forward = decimation in frequency (natural in, digit-reversed out),
// inverse = decimation in time with the stages mirrored (digit-reversed in, natural out).
struct AxisPlan {
    int M;                  // transform length
    int logM;
    int nst;                // number of stages
    int radix[kMaxStages];  // product = M, each in {8, 4, 2}
};

// device-resident index tables of one axis
struct AxisTables {
    const uint16_t* perm;     // position p after the forward stages holds frequency perm[p]
    const uint16_t* invperm;  // frequency k sits at position invperm[k]
};

// Per-member scalars as the kernels read them.
struct DevMember {
    double G11, Gt, Gm;      // Gt = G44 + G44', Gm = G12 + G44 - G44' (Eq. 4 expanded, O2)
    double escale;           // 1 / (eps0 * epsB)   (Eq. 6 prefactor)
    double L;
    double Eext[3];
    // time-dependent excitation: E_ext(t) = Eext + wamp sin(womega t + wphase) when wave != 0
    double wamp[3], womega, wphase;
    int32_t wave, pad;
};

struct DevLandau {
    double a1[3];
    double a11, a12, a111, a112, a123;
    double a1111, a1112, a1122, a1123;
    int32_t active;
    int32_t pad;
};

struct Geometry {
    int n[3];          // nx ny nz
    int m[3];          // padded box
    int periodic[3];
    int images[3];
    double d[3];
    int zero_mode;
    int Lx;            // m[0]/2 + 1 complex points per spectrum row
    int pitch;         // row pitch of the spectra (complex elements), multiple of the lane tile
    int pitch64;       // same for the fp64 precompute spectra
    int lanes;         // kx lanes per block in the strided passes (128 B of complex numbers)
    int lanes64;
};

// ---- launchers (fe_fft.cu) --------------------------------------------------------------------
struct FftCtx {
    const void* tw;           // cx<T>[kTwiddleN]
    AxisPlan plan[3];         // [0]: x (length m_x/2 complex), [1]: y, [2]: z
    AxisTables tab[3];
};

// real rows -> half spectrum rows.  in: T real rows of n_in valid reals (zero-padded to 2*plan.M),
// out: complex rows of pitch `pitch` holding plan.M + 1 entries.
template <typename T>
cudaError_t launch_xfwd(const FftCtx& c, const T* in, void* out, int n_in, int rows_per_slab, int slabs,
                        int64_t in_row_stride, int64_t in_slab_stride, int64_t out_row_stride,
                        int64_t out_slab_stride, cudaStream_t st);
template <typename T>
cudaError_t launch_xinv(const FftCtx& c, const void* in, T* out, int n_out, int rows_per_slab, int slabs,
                        int64_t in_row_stride, int64_t in_slab_stride, int64_t out_row_stride,
                        int64_t out_slab_stride, cudaStream_t st);
// strided pass along one axis (axis = 1 or 2 picks plan/tables): forward reads n_keep rows and writes
// plan.M rows (natural frequency order); inverse reads plan.M rows and writes n_keep rows.
template <typename T>
cudaError_t launch_axis(const FftCtx& c, int axis, int dir, const void* in, void* out, int n_keep,
                        int lanes, int pitch_used, int outer, int batch, int64_t in_sa, int64_t in_so,
                        int64_t in_sb, int64_t out_sa, int64_t out_so, int64_t out_sb, cudaStream_t st);
// fused z-forward, K multiply, z-inverse, in place on S[b][3][nz][My][pitch]
template <typename T>
cudaError_t launch_zmul(const FftCtx& c, void* S, const T* Kt, const DevMember* members, int nz, int My,
                        int lanes, int pitch, int batch, cudaStream_t st);
// complex fp64 box spectrum -> real octant table of T (scaled)
template <typename T>
cudaError_t launch_extract(const void* Sbox, T* Kt_comp, int Mz, int My, int Lx, int pitch64, int pitchT,
                           double scale, int lanes, int64_t k_skz, int64_t k_sky, int64_t k_sg, cudaStream_t st);
size_t zmul_smem_bytes(int Mz, int lanes, size_t cx_bytes);

// ---- size-specialised register FFT passes (fe_fft2_*.cu); same data layouts as the generic launchers above
bool x2_supported(int Mc);
bool axis2_supported(int M);
bool zmul2_supported(int M);
template <typename T>
cudaError_t launch_xfwd2(const FftCtx& c, const T* in, void* out, int n_real, int64_t nrows, int64_t real_rs,
                         const int64_t spec[4] /* ny, s_plane, s_row, s_g */, int lanes, cudaStream_t st);
template <typename T>
cudaError_t launch_xinv2(const FftCtx& c, const void* in, T* out, int n_real, int64_t nrows, int64_t real_rs,
                         const int64_t spec[4], int lanes, cudaStream_t st);
template <typename T>
cudaError_t launch_xinv2_slab(const FftCtx& c, const void* in, T* out, int n_real, int comps, int ny, int nz, int zb, int zn,
                              const int64_t spec[4], int lanes, cudaStream_t st);
bool xinv_slab_supported(int Mc, int n_real, int ny, int lanes, size_t elem);
template <typename T>
cudaError_t launch_axis2(const FftCtx& c, int axis, int dir, const void* in, void* out, int n_keep, int n0, int n1,
                         int batch, int64_t in_sa, int64_t in_s0, int64_t in_s1, int64_t in_sb, int64_t out_sa,
                         int64_t out_s0, int64_t out_s1, int64_t out_sb, cudaStream_t st);
bool axis4_supported(int M);
int axis4_slot(int M, int k);
void axis4_radices(int M, int r[3]);
template <typename T>
cudaError_t launch_axis4(const FftCtx& c, int axis, int dir, const void* in, void* out, int n_keep, int n0, int n1,
                         int batch, int64_t in_s0, int64_t in_s1, int64_t in_sb, int64_t out_s0, int64_t out_s1,
                         int64_t out_sb, cudaStream_t st);
template <typename T>
cudaError_t launch_zmul2(const FftCtx& c, void* S, const T* Kt, const DevMember* members, int nz, int My, int ngroups,
                         int batch, const int64_t sstr[4] /* cs, s_z, s_ky, s_g */,
                         const int64_t kstr[4] /* kcs, k_skz, k_sky, k_sg */,
                         const int perm[3] /* slot-order radices of ky, {0,0,0}: natural */, cudaStream_t st);
// x and y passes fused through an L2-resident ring of S1 planes (fe_fft2_xy.cu).  counters: 2 * nplanes + 1 ints.
bool xy_supported(int Mx, int My, int nx, int ny);
template <typename T>
cudaError_t launch_xyfwd(const FftCtx& c, const T* P, void* ring, void* S2, int nx, int ny, int nz, int nplanes, int G,
                         int ring_slots, int64_t s2_sz, int64_t s2_sg, int64_t s2_sb, int* counters, cudaStream_t st);
cudaError_t fft_configure();     // raise dynamic shared memory limits; call once

// ---- tensor (fe_tensor.cu) --------------------------------------------------------------------
cudaError_t tensor_init_tables();
// real-space kernel of one component on the circular box [mz][my][mx] (fp64)
cudaError_t launch_tensor_box(const Geometry& g, double* box6 /* [6][mz][my][mx] or one comp */,
                              int comp_first, int ncomp, cudaStream_t st);
cudaError_t launch_zero_mode(const Geometry& g, double* box, int comp, double* scratch /* one device double */,
                             cudaStream_t st);

// ---- local terms (fe_local.cu) ----------------------------------------------------------------
struct LocalArgs {
    const void* Y;        // state the RHS is evaluated at           [B][3][N]
    const void* Eelec;    // electrostatic field (may be null)       [B][3][N]
    const void* baseY;    // Yout = baseY + cy * k  (null: Yout = cy * k)
    void* Yout;
    const void* accIn;    // accOut = accIn + ca * k (both null: skipped)
    void* accOut;
    double cy, ca;
    // stage combinations of the multistep / embedded integrators folded into the same epilogue:
    //   kOut = k (raw right-hand side, may be null);  Yout = baseY + sum_{j < nlin} lc[j] * lk[j] + cy * k
    void* kOut;
    const void* lk[4];
    double lc[4];
    int nlin;
    const uint8_t* map;   // null: material 0 everywhere
    const DevLandau* mats;    // [B][nmat]
    const DevMember* members; // [B]
    int nmat;
    int n[3];
    int periodic[3];
    double d[3];
    uint32_t terms;
    int batch;
    int mixed;            // any member has Gm != 0
    int vac0;             // material 0 of some member is vacuum (matters without a map: that member is all vacuum)
    double t;             // time at which E_ext is sampled (stage time)
    // filled by launch_local
    double id2[3];        // 1 / D_a^2
    double i4[3];         // 1 / (4 D_x D_y), 1 / (4 D_x D_z), 1 / (4 D_y D_z)
    int zchunk;           // planes per block
    // z slab of this launch (FE_OPT_XL_SLABS: the x inverse pass hands E_elec to the local step slab by slab through the
    // first planes of every component's region of the E buffer, which stay in L2).  zend == 0: all planes
    int zbeg, zend;
    int e_z0;             // Eelec holds plane z of a component at plane z - e_z0 of its region (0: the whole field)
};
template <typename T> cudaError_t launch_local(const LocalArgs& a, cudaStream_t st);

struct EnergyArgs {
    const void* P;
    const void* Eelec;
    const uint8_t* map;
    const DevLandau* mats;
    const DevMember* members;
    int nmat;
    int n[3];
    int periodic[3];
    double d[3];
    uint32_t terms;
    int batch;
    double t;             // time at which E_ext is sampled
    double* partials;     // [B][nblk][8]
    double* out;          // [B][8] device
    int nblk;
};
template <typename T> cudaError_t launch_energy(const EnergyArgs& a, cudaStream_t st);

// ---- integrator array kernels (fe_integ.cu) ---------------------------------------------------
struct LinArgs {
    const void* k[6];
    double c[6];
};
// y5 = P + sum_j b5.c_j k_j;  *err (device double, reset here) = max_i |sum_j d.c_j k_j[i]|
template <typename T>
cudaError_t launch_rk45_final(T* y5, const T* P, const LinArgs& b5, const LinArgs& d, int64_t n, double* err, cudaStream_t st);

}  // namespace fe
