// fe_api.cu -- the C ABI of libfe_b200 (include/fe.h): argument checking, workspace layout, the
// sequence of kernel launches of one RHS evaluation and the explicit
// integrators (a5).  All arithmetic of the method is in the kernels.
#include "../../include/fe.h"
#include "fe_internal.h"

#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include <vector>

using namespace fe;

static thread_local char g_err[512] = "";

static fe_status fail(fe_status s, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return s;
}

#define FE_CUDA(call)                                                                          \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess) return fail(FE_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
    } while (0)

static size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

struct fe_grid {
    fe_grid_desc desc;
    Geometry geo;
    bool f32;
    size_t rsz, csz;                 // bytes of a real / complex element of the state dtype
    int64_t N;
    // host mirrors of the coefficient tables
    std::vector<DevLandau> h_mats;   // [B][nmat]
    std::vector<uint8_t> mat_set;
    std::vector<DevMember> h_members;
    std::vector<fe_global> h_globals;
    std::vector<uint8_t> glob_set;
    bool dirty;
    int mixed;
    // small device tables owned by the library
    unsigned char* d_small;
    DevLandau* d_mats;
    DevMember* d_members;
    double* d_eout;
    FftCtx ctx;                      // state dtype
    FftCtx ctx64;                    // fp64 (tensor precompute)
    const uint8_t* map;
    // workspace (borrowed)
    unsigned char* ws;
    size_t ws_bytes;
    size_t o_Kt, o_S1, o_S2, o_E, o_Y, o_ACC, o_PP, o_K[6], o_part, o_cnt, o_box, o_Sbox, total_bytes;
    int vac0;                        // material 0 of some member is vacuum
    int opt_fuse_xy;                 // FE_OPT_FUSE_XY
    int opt_xl_slabs;                // FE_OPT_XL_SLABS
    int opt_xy_ring;                 // FE_OPT_XY_RING (0: automatic)
    int nblk;
    bool tensor_ready;
    bool fast[3];                    // size-specialised register FFT kernels available for the x / y / z pass
    bool tiled;                      // spectra and tensor table in the tiled layouts (all three passes fast)
    uint64_t launches;
    // optional per-kernel CUDA-event timing (fe_profile): event i precedes the launch of kind prof_kind[i]
    // CUDA-graph replay of fe_step (one captured unit of steps, replayed on an internal stream)
    cudaStream_t gstream;
    cudaEvent_t gev_in, gev_out;
    cudaGraphExec_t gexec;
    bool gvalid, goff;               // cached graph usable / graphs disabled for this grid after a failure
    void* gP; double gdt; int ginteg; uint32_t gterms; uint64_t gunit_launches;
    double time;                     // simulation time (advanced by fe_step / fe_step_rk45); E_ext(t) is sampled from it
    double tstage;                   // time of the stage being evaluated
    bool any_wave;                   // some member has a time-dependent excitation: no graph replay
    bool prof_on;
    std::vector<cudaEvent_t> prof_ev;
    std::vector<int> prof_kind;
    size_t prof_used;
};

enum { K_XFWD = 0, K_YFWD, K_ZMUL, K_YINV, K_XINV, K_LOCAL, K_OTHER, K_XYFWD, K_XYINV, K_NKINDS };

// record an event on the stream before a launch of `kind` (kind < 0: closes the previous interval)
static void mark(fe_grid* g, int kind, cudaStream_t st)
{
    if (!g->prof_on) return;
    if (g->prof_used >= 60000) return;
    if (g->prof_used == g->prof_ev.size()) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) return;
        g->prof_ev.push_back(e);
        g->prof_kind.push_back(-1);
    }
    cudaEventRecord(g->prof_ev[g->prof_used], st);
    g->prof_kind[g->prof_used] = kind;
    ++g->prof_used;
}

static AxisPlan make_plan(int M)
{
    AxisPlan p;
    memset(&p, 0, sizeof(p));
    p.M = M;
    int L = 0;
    while ((1 << L) < M) ++L;
    p.logM = L;
    int n8 = L / 3, rem = L % 3, k = 0;
    if (rem == 1 && n8 >= 1) {
        for (int i = 0; i < n8 - 1; ++i) p.radix[k++] = 8;
        p.radix[k++] = 4;
        p.radix[k++] = 4;
    } else {
        for (int i = 0; i < n8; ++i) p.radix[k++] = 8;
        if (rem == 2) p.radix[k++] = 4;
        if (rem == 1) p.radix[k++] = 2;
    }
    p.nst = k;
    return p;
}

// position p after the forward (DIF) stages holds frequency perm[p]:
// p = q1 * M/R1 + q2 * M/(R1 R2) + ...,  k = q1 + R1 (q2 + R2 (q3 + ...))
static void make_perm(const AxisPlan& pl, std::vector<uint16_t>& perm, std::vector<uint16_t>& inv)
{
    perm.assign(pl.M, 0);
    inv.assign(pl.M, 0);
    for (int p = 0; p < pl.M; ++p) {
        int rem = p, span = pl.M, k = 0, w = 1;
        for (int st = 0; st < pl.nst; ++st) {
            span /= pl.radix[st];
            int q = rem / span;
            rem -= q * span;
            k += q * w;
            w *= pl.radix[st];
        }
        perm[p] = (uint16_t)k;
        inv[k] = (uint16_t)p;
    }
}

static bool pow2_in(int v, int lo, int hi) { return v >= lo && v <= hi && (v & (v - 1)) == 0; }

extern "C" const char* fe_last_error(void) { return g_err; }
extern "C" const char* fe_version(void) { return "fe_b200 0.1 (sm_100a)"; }

static void layout_workspace(fe_grid* g)
{
    const Geometry& q = g->geo;
    const int B = g->desc.batch;
    const int Hy = q.m[1] / 2 + 1, Hz = q.m[2] / 2 + 1;
    size_t off = 0;
    g->o_Kt = off;  off += align_up((size_t)6 * Hz * Hy * q.pitch * g->rsz);
    const size_t hot0 = off;
    g->o_S1 = off;  off += align_up((size_t)B * 3 * q.n[2] * q.n[1] * q.pitch * g->csz);
    g->o_S2 = off;  off += align_up((size_t)B * 3 * q.n[2] * q.m[1] * q.pitch * g->csz);
    g->o_E = off;   off += align_up((size_t)B * 3 * g->N * g->rsz);
    g->o_Y = off;   off += align_up((size_t)B * 3 * g->N * g->rsz);
    g->o_ACC = off; off += align_up((size_t)B * 3 * g->N * g->rsz);
    g->o_PP = off;  off += align_up((size_t)B * 3 * g->N * g->rsz);
    for (int j = 0; j < 6; ++j) { g->o_K[j] = off; off += align_up((size_t)B * 3 * g->N * g->rsz); }   // RK45 / AB3M2 stages
    const size_t hot1 = off;
    // precompute scratch overlays the hot region (the tensor is computed before any step)
    size_t s = hot0;
    g->o_box = s;   s += align_up((size_t)q.m[0] * q.m[1] * q.m[2] * sizeof(double));
    g->o_Sbox = s;  s += align_up((size_t)q.m[2] * q.m[1] * q.pitch64 * 2 * sizeof(double));
    off = hot1 > s ? hot1 : s;
    g->nblk = 296;
    g->o_part = off; off += align_up((size_t)B * g->nblk * 8 * sizeof(double));
    g->o_cnt = off;  off += align_up(((size_t)2 * B * 3 * q.n[2] + 1) * sizeof(int));     // plane counters of the fused x+y pass
    g->total_bytes = off;
}

extern "C" fe_status fe_create_grid(const fe_grid_desc* d, fe_grid** out)
{
    if (!d || !out) return fail(FE_EINVAL, "null argument");
    const int n[3] = {d->nx, d->ny, d->nz};
    const double dd[3] = {d->dx, d->dy, d->dz};
    for (int a = 0; a < 3; ++a) {
        if (d->periodic[a] == 1) {
            if (!pow2_in(n[a], 4, 1024))
                return fail(FE_EINVAL, "n[%d] = %d: a periodic axis must be a power of two in [4, 1024]", a, n[a]);
        } else {
            // open axis: zero-padded to the next power of two >= 2 n, any length goes (x even: the R2C pass packs pairs)
            if (n[a] < 2 || n[a] > 512) return fail(FE_EINVAL, "n[%d] = %d: an open axis must have 2..512 cells", a, n[a]);
            if (a == 0 && (n[a] & 1)) return fail(FE_EINVAL, "n[0] = %d: an open x axis must have an even number of cells", n[a]);
        }
        if (!(dd[a] > 0.0) || !isfinite(dd[a])) return fail(FE_EINVAL, "cell size d[%d] must be > 0", a);
        if (d->periodic[a] != 0 && d->periodic[a] != 1) return fail(FE_EINVAL, "periodic[%d] must be 0 or 1", a);
        if (d->pbc_images[a] < 0 || d->pbc_images[a] > 64) return fail(FE_EINVAL, "pbc_images[%d] out of range", a);
    }
    if (d->batch < 1 || d->batch > 16384) return fail(FE_EINVAL, "batch must be in [1, 16384]");
    if (d->dtype != FE_F64 && d->dtype != FE_F32) return fail(FE_EINVAL, "dtype must be FE_F64 or FE_F32");
    if (d->n_materials < 1 || d->n_materials > 255) return fail(FE_EINVAL, "n_materials must be in [1, 255]");
    if ((int64_t)d->batch * 3 * d->nz > 0x7fffffffLL) return fail(FE_EINVAL, "batch * nz too large");

    fe_grid* g = new (std::nothrow) fe_grid();
    if (!g) return fail(FE_ENOMEM, "host allocation failed");
    g->desc = *d;
    g->f32 = d->dtype == FE_F32;
    g->rsz = g->f32 ? 4 : 8;
    g->csz = 2 * g->rsz;
    g->N = (int64_t)d->nx * d->ny * d->nz;
    Geometry& q = g->geo;
    for (int a = 0; a < 3; ++a) {
        q.n[a] = n[a];
        q.periodic[a] = d->periodic[a];
        q.images[a] = d->periodic[a] ? d->pbc_images[a] : 0;
        q.m[a] = n[a];
        if (!d->periodic[a]) { q.m[a] = 4; while (q.m[a] < 2 * n[a]) q.m[a] *= 2; }
        q.d[a] = dd[a];
    }
    q.zero_mode = d->zero_mode;
    q.Lx = q.m[0] / 2 + 1;
    // lanes: 128 bytes of complex numbers, halved until the fused z tile (3 components) fits in shared memory
    auto pick_lanes = [&](size_t cxb) {
        int l = (int)(128 / cxb);
        while (l > 1 && zmul_smem_bytes(q.m[2], l, cxb) > 200 * 1024) l >>= 1;
        while (l > 1 && (size_t)q.m[1] * l * cxb > 200 * 1024) l >>= 1;
        return l;
    };
    q.lanes = pick_lanes(g->csz);
    q.lanes64 = pick_lanes(16);
    const int pl = (int)(128 / g->csz);
    q.pitch = (q.Lx + pl - 1) / pl * pl;
    q.pitch64 = (q.Lx + 7) / 8 * 8;
    {
        // size-specialised register passes per axis; any other transform length takes the generic shared-memory pass
        const size_t lanes_full = 128 / g->csz;
        g->fast[0] = x2_supported(q.m[0] / 2);
        g->fast[1] = axis2_supported(q.m[1]) && (size_t)q.lanes == lanes_full;
        g->fast[2] = zmul2_supported(q.m[2]) && (size_t)q.lanes == lanes_full;
        // Tiled layouts (L = 128 bytes of consecutive kx, G = pitch / L groups), used when every pass is fast:
        //   S1[b][c][z][g][y][L]   the y pass reads / writes whole contiguous tiles,
        //   S2[b][c][g][z][ky][L]  likewise (ky in slot order when the bulk-copy y pass runs); the fused z pass reads
        //                          128-byte rows 64 KB apart instead of 2 MB apart,
        //   Kt[6][g][ky][kz][L]    its tensor tile is contiguous too.
        // otherwise the spectra stay row-major (the kernels take strides, both layouts run the same code).
        g->tiled = g->fast[0] && g->fast[1] && g->fast[2];
    }
    g->dirty = true;
    g->mixed = 0;
    g->vac0 = 0;
    g->opt_fuse_xy = 0;
    g->opt_xl_slabs = 0;
    g->opt_xy_ring = 0;
    g->map = nullptr;
    g->ws = nullptr;
    g->ws_bytes = 0;
    g->tensor_ready = false;
    g->launches = 0;
    g->prof_on = false;
    g->prof_used = 0;
    g->time = 0.0; g->tstage = 0.0; g->any_wave = false;
    g->gstream = nullptr; g->gev_in = nullptr; g->gev_out = nullptr; g->gexec = nullptr;
    g->gvalid = false; g->goff = false; g->gP = nullptr; g->gdt = 0.0; g->ginteg = -1; g->gterms = 0; g->gunit_launches = 0;
    const int B = d->batch, M = d->n_materials;
    g->h_mats.assign((size_t)B * M, DevLandau{});
    g->mat_set.assign((size_t)B * M, 0);
    g->h_members.assign(B, DevMember{});
    g->h_globals.assign(B, fe_global{});
    g->glob_set.assign(B, 0);
    layout_workspace(g);

    // small device tables: twiddles (fp64 + fp32), perm/invperm per axis, coefficient tables, energy out
    AxisPlan plans[3] = {make_plan(q.m[0] / 2), make_plan(q.m[1]), make_plan(q.m[2])};
    std::vector<uint16_t> perm[3], inv[3];
    for (int a = 0; a < 3; ++a) make_perm(plans[a], perm[a], inv[a]);
    size_t off = 0;
    const size_t o_tw64 = off; off += align_up(kTwiddleN * 16);
    const size_t o_tw32 = off; off += align_up(kTwiddleN * 8);
    size_t o_perm[3], o_inv[3];
    for (int a = 0; a < 3; ++a) {
        o_perm[a] = off; off += align_up(plans[a].M * 2);
        o_inv[a] = off;  off += align_up(plans[a].M * 2);
    }
    const size_t o_mats = off; off += align_up((size_t)B * M * sizeof(DevLandau));
    const size_t o_mem = off;  off += align_up((size_t)B * sizeof(DevMember));
    const size_t o_eout = off; off += align_up((size_t)B * 8 * sizeof(double));
    std::vector<unsigned char> h(off, 0);
    {
        const long double twopi = 6.283185307179586476925286766559005768L;
        double* t64 = reinterpret_cast<double*>(h.data() + o_tw64);
        float* t32 = reinterpret_cast<float*>(h.data() + o_tw32);
        for (int k = 0; k < kTwiddleN; ++k) {
            const long double ang = twopi * k / kTwiddleN;
            const long double c = (k == kTwiddleN / 4 || k == 3 * kTwiddleN / 4) ? 0.0L : cosl(ang);
            const long double s = (k == 0 || k == kTwiddleN / 2) ? 0.0L : sinl(ang);
            t64[2 * k] = (double)c;  t64[2 * k + 1] = (double)(-s);
            t32[2 * k] = (float)c;   t32[2 * k + 1] = (float)(-s);
        }
        for (int a = 0; a < 3; ++a) {
            memcpy(h.data() + o_perm[a], perm[a].data(), plans[a].M * 2);
            memcpy(h.data() + o_inv[a], inv[a].data(), plans[a].M * 2);
        }
    }
    cudaError_t e = cudaMalloc(&g->d_small, off);
    if (e != cudaSuccess) { delete g; return fail(FE_ECUDA, "cudaMalloc(tables): %s", cudaGetErrorString(e)); }
    e = cudaMemcpy(g->d_small, h.data(), off, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = fft_configure();
    if (e == cudaSuccess) e = tensor_init_tables();
    if (e != cudaSuccess) {
        cudaFree(g->d_small);
        delete g;
        return fail(FE_ECUDA, "table setup: %s", cudaGetErrorString(e));
    }
    g->d_mats = reinterpret_cast<DevLandau*>(g->d_small + o_mats);
    g->d_members = reinterpret_cast<DevMember*>(g->d_small + o_mem);
    g->d_eout = reinterpret_cast<double*>(g->d_small + o_eout);
    for (int a = 0; a < 3; ++a) {
        g->ctx.plan[a] = g->ctx64.plan[a] = plans[a];
        g->ctx.tab[a].perm = g->ctx64.tab[a].perm = reinterpret_cast<const uint16_t*>(g->d_small + o_perm[a]);
        g->ctx.tab[a].invperm = g->ctx64.tab[a].invperm = reinterpret_cast<const uint16_t*>(g->d_small + o_inv[a]);
    }
    g->ctx64.tw = g->d_small + o_tw64;
    g->ctx.tw = g->f32 ? g->d_small + o_tw32 : g->d_small + o_tw64;
    *out = g;
    return FE_OK;
}

extern "C" fe_status fe_destroy_grid(fe_grid* g)
{
    if (!g) return FE_OK;
    for (cudaEvent_t e : g->prof_ev) cudaEventDestroy(e);
    if (g->gexec) cudaGraphExecDestroy(g->gexec);
    if (g->gev_in) cudaEventDestroy(g->gev_in);
    if (g->gev_out) cudaEventDestroy(g->gev_out);
    if (g->gstream) cudaStreamDestroy(g->gstream);
    cudaFree(g->d_small);
    delete g;
    return FE_OK;
}

extern "C" size_t fe_workspace_bytes(const fe_grid* g) { return g ? g->total_bytes : 0; }

extern "C" fe_status fe_padded_dims(const fe_grid* g, int32_t out[3])
{
    if (!g || !out) return fail(FE_EINVAL, "null argument");
    for (int a = 0; a < 3; ++a) out[a] = g->geo.m[a];
    return FE_OK;
}

extern "C" uint64_t fe_launch_count(const fe_grid* g) { return g ? g->launches : 0; }

extern "C" fe_status fe_bind_workspace(fe_grid* g, void* dev, size_t bytes)
{
    if (!g || !dev) return fail(FE_EINVAL, "null argument");
    if (bytes < g->total_bytes) return fail(FE_ENOMEM, "workspace of %zu bytes given, %zu needed", bytes, g->total_bytes);
    if (reinterpret_cast<uintptr_t>(dev) % 256) return fail(FE_EINVAL, "workspace must be 256-byte aligned");
    g->ws = static_cast<unsigned char*>(dev);
    g->ws_bytes = bytes;
    g->tensor_ready = false;
    g->gvalid = false;
    return FE_OK;
}

extern "C" fe_status fe_set_material(fe_grid* g, int32_t member, int32_t id, const fe_landau* m)
{
    if (!g || !m) return fail(FE_EINVAL, "null argument");
    const int B = g->desc.batch, M = g->desc.n_materials;
    if (member < -1 || member >= B) return fail(FE_EINVAL, "member %d out of range", member);
    if (id < 0 || id >= M) return fail(FE_EINVAL, "material id %d out of range", id);
    const double* v = &m->a1[0];
    for (int i = 0; i < 12; ++i)
        if (!isfinite(v[i])) return fail(FE_EINVAL, "non-finite Landau coefficient");
    DevLandau dl;
    memset(&dl, 0, sizeof(dl));
    for (int i = 0; i < 3; ++i) dl.a1[i] = m->a1[i];
    dl.a11 = m->a11; dl.a12 = m->a12; dl.a111 = m->a111; dl.a112 = m->a112; dl.a123 = m->a123;
    dl.a1111 = m->a1111; dl.a1112 = m->a1112; dl.a1122 = m->a1122; dl.a1123 = m->a1123;
    dl.active = m->active ? 1 : 0;
    for (int b = (member < 0 ? 0 : member); b < (member < 0 ? B : member + 1); ++b) {
        g->h_mats[(size_t)b * M + id] = dl;
        g->mat_set[(size_t)b * M + id] = 1;
    }
    g->dirty = true;
    return FE_OK;
}

extern "C" fe_status fe_set_global(fe_grid* g, int32_t member, const fe_global* gl)
{
    if (!g || !gl) return fail(FE_EINVAL, "null argument");
    const int B = g->desc.batch;
    if (member < -1 || member >= B) return fail(FE_EINVAL, "member %d out of range", member);
    if (!(gl->eps0 > 0.0) || !(gl->epsB > 0.0) || !isfinite(gl->eps0 * gl->epsB))
        return fail(FE_EINVAL, "eps0 and epsB must be > 0");
    if (!isfinite(gl->G11) || !isfinite(gl->G12) || !isfinite(gl->G44) || !isfinite(gl->G44p) || !isfinite(gl->L))
        return fail(FE_EINVAL, "non-finite coefficient");
    for (int b = (member < 0 ? 0 : member); b < (member < 0 ? B : member + 1); ++b) {
        DevMember& dm = g->h_members[b];
        dm.G11 = gl->G11;
        dm.Gt = gl->G44 + gl->G44p;
        dm.Gm = gl->G12 + gl->G44 - gl->G44p;
        dm.escale = 1.0 / (gl->eps0 * gl->epsB);
        dm.L = gl->L;
        g->h_globals[b] = *gl;
        g->glob_set[b] = 1;
    }
    g->dirty = true;
    return FE_OK;
}

extern "C" fe_status fe_set_external_field(fe_grid* g, int32_t member, const double E[3])
{
    if (!g || !E) return fail(FE_EINVAL, "null argument");
    const int B = g->desc.batch;
    if (member < -1 || member >= B) return fail(FE_EINVAL, "member %d out of range", member);
    for (int i = 0; i < 3; ++i)
        if (!isfinite(E[i])) return fail(FE_EINVAL, "non-finite field");
    for (int b = (member < 0 ? 0 : member); b < (member < 0 ? B : member + 1); ++b)
        for (int i = 0; i < 3; ++i) g->h_members[b].Eext[i] = E[i];
    g->dirty = true;
    return FE_OK;
}

extern "C" fe_status fe_set_external_wave(fe_grid* g, int32_t member, const double amp[3], double omega, double phase)
{
    if (!g || !amp) return fail(FE_EINVAL, "null argument");
    const int B = g->desc.batch;
    if (member < -1 || member >= B) return fail(FE_EINVAL, "member %d out of range", member);
    if (!isfinite(amp[0]) || !isfinite(amp[1]) || !isfinite(amp[2]) || !isfinite(omega) || !isfinite(phase))
        return fail(FE_EINVAL, "non-finite wave parameter");
    const bool on = amp[0] != 0.0 || amp[1] != 0.0 || amp[2] != 0.0;
    for (int b = (member < 0 ? 0 : member); b < (member < 0 ? B : member + 1); ++b) {
        DevMember& dm = g->h_members[b];
        for (int i = 0; i < 3; ++i) dm.wamp[i] = amp[i];
        dm.womega = omega;
        dm.wphase = phase;
        dm.wave = on ? 1 : 0;
    }
    g->dirty = true;
    return FE_OK;
}

extern "C" fe_status fe_set_time(fe_grid* g, double t)
{
    if (!g || !isfinite(t)) return fail(FE_EINVAL, "bad argument");
    g->time = t;
    return FE_OK;
}

extern "C" fe_status fe_get_time(const fe_grid* g, double* t)
{
    if (!g || !t) return fail(FE_EINVAL, "null argument");
    *t = g->time;
    return FE_OK;
}

extern "C" fe_status fe_set_material_map(fe_grid* g, const uint8_t* dev_map)
{
    if (!g) return fail(FE_EINVAL, "null argument");
    g->map = dev_map;
    g->gvalid = false;
    return FE_OK;
}

extern "C" fe_status fe_set_option(fe_grid* g, int32_t option, int32_t value)
{
    if (!g) return fail(FE_EINVAL, "null argument");
    if (option == FE_OPT_FUSE_XY && (value == 0 || value == 1)) {
        g->opt_fuse_xy = value;
        g->gvalid = false;               // a captured graph holds the other kernels
        return FE_OK;
    }
    if (option == FE_OPT_XY_RING && value >= 0 && value <= 4096) {
        g->opt_xy_ring = value;
        g->gvalid = false;
        return FE_OK;
    }
    if (option == FE_OPT_XL_SLABS && value >= 0 && value <= 64) {
        g->opt_xl_slabs = value;
        g->gvalid = false;
        return FE_OK;
    }
    return fail(FE_EINVAL, "unknown option %d or bad value %d", option, value);
}

extern "C" fe_status fe_get_option(fe_grid* g, int32_t option, int32_t* value)
{
    if (!g || !value) return fail(FE_EINVAL, "null argument");
    if (option == FE_OPT_FUSE_XY) { *value = g->opt_fuse_xy; return FE_OK; }
    if (option == FE_OPT_XY_RING) { *value = g->opt_xy_ring; return FE_OK; }
    if (option == FE_OPT_XL_SLABS) { *value = g->opt_xl_slabs; return FE_OK; }
    if (option == FE_OPT_XY_TIMEOUTS) {
        *value = 0;
        if (!g->ws) return FE_OK;
        int flag = 0;
        FE_CUDA(cudaDeviceSynchronize());
        const int nplanes = g->desc.batch * 3 * g->geo.n[2];
        FE_CUDA(cudaMemcpy(&flag, g->ws + g->o_cnt + (size_t)2 * nplanes * sizeof(int), sizeof(int), cudaMemcpyDeviceToHost));
        *value = flag != 0;
        return FE_OK;
    }
    return fail(FE_EINVAL, "unknown option %d", option);
}

static fe_status sync_params(fe_grid* g, cudaStream_t st)
{
    const int B = g->desc.batch, M = g->desc.n_materials;
    for (int b = 0; b < B; ++b) {
        if (!g->glob_set[b]) return fail(FE_ESTATE, "fe_set_global was not called for member %d", b);
        for (int m = 0; m < M; ++m)
            if (!g->mat_set[(size_t)b * M + m]) return fail(FE_ESTATE, "material %d of member %d is unset", m, b);
    }
    if (!g->dirty) return FE_OK;
    g->gvalid = false;               // kernel variants (mixed term) may change with the coefficients
    g->mixed = 0;
    g->vac0 = 0;
    g->any_wave = false;
    for (int b = 0; b < B; ++b) {
        if (g->h_members[b].Gm != 0.0) g->mixed = 1;
        if (!g->h_mats[(size_t)b * M].active) g->vac0 = 1;
        if (g->h_members[b].wave) g->any_wave = true;
    }
    FE_CUDA(cudaMemcpyAsync(g->d_mats, g->h_mats.data(), (size_t)B * M * sizeof(DevLandau), cudaMemcpyHostToDevice, st));
    FE_CUDA(cudaMemcpyAsync(g->d_members, g->h_members.data(), (size_t)B * sizeof(DevMember), cudaMemcpyHostToDevice, st));
    // pageable host memory: the copies are staged before the calls return, the vectors may change afterwards
    g->dirty = false;
    return FE_OK;
}

// ---- a0 ------------------------------------------------------------------------------------------
template <typename T>
static fe_status precompute_T(fe_grid* g, cudaStream_t st)
{
    const Geometry& q = g->geo;
    double* box = reinterpret_cast<double*>(g->ws + g->o_box);
    void* Sbox = g->ws + g->o_Sbox;
    T* Kt = reinterpret_cast<T*>(g->ws + g->o_Kt);
    const int Hy = q.m[1] / 2 + 1, Hz = q.m[2] / 2 + 1;
    const double scale = 1.0 / ((double)(q.m[0] / 2) * q.m[1] * q.m[2]);
    const int64_t p64 = q.pitch64;
    for (int c = 0; c < 6; ++c) {
        FE_CUDA(launch_tensor_box(q, box, c, 1, st));
        FE_CUDA(launch_zero_mode(q, box, c, g->d_eout, st));
        FE_CUDA(launch_xfwd<double>(g->ctx64, box, Sbox, q.m[0], q.m[1], q.m[2], q.m[0], (int64_t)q.m[0] * q.m[1],
                                    p64, p64 * q.m[1], st));
        FE_CUDA(launch_axis<double>(g->ctx64, 1, -1, Sbox, Sbox, q.m[1], q.lanes64, q.pitch64, q.m[2], 1, p64,
                                    p64 * q.m[1], 0, p64, p64 * q.m[1], 0, st));
        FE_CUDA(launch_axis<double>(g->ctx64, 2, -1, Sbox, Sbox, q.m[2], q.lanes64, q.pitch64, q.m[1], 1,
                                    p64 * q.m[1], p64, 0, p64 * q.m[1], p64, 0, st));
        const int L = (int)(128 / g->csz);
        if (g->tiled)
            FE_CUDA(launch_extract<T>(Sbox, Kt + (int64_t)c * Hz * Hy * q.pitch, q.m[2], q.m[1], q.Lx, q.pitch64, q.pitch,
                                      scale, L, L, (int64_t)Hz * L, (int64_t)Hy * Hz * L, st));
        else
            FE_CUDA(launch_extract<T>(Sbox, Kt + (int64_t)c * Hz * Hy * q.pitch, q.m[2], q.m[1], q.Lx, q.pitch64, q.pitch,
                                      scale, L, (int64_t)Hy * q.pitch, q.pitch, L, st));
        g->launches += 5 + ((q.zero_mode && q.periodic[0] + q.periodic[1] + q.periodic[2] == 2) ? 1 : 0);
    }
    return FE_OK;
}

extern "C" fe_status fe_precompute_tensor(fe_grid* g, void* stream)
{
    if (!g) return fail(FE_EINVAL, "null argument");
    if (!g->ws) return fail(FE_ESTATE, "no workspace bound");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    fe_status s = g->f32 ? precompute_T<float>(g, st) : precompute_T<double>(g, st);
    if (s != FE_OK) return s;
    FE_CUDA(cudaStreamSynchronize(st));
    g->tensor_ready = true;
    return FE_OK;
}

extern "C" fe_status fe_get_tensor(fe_grid* g, double* host_out, void* stream)
{
    if (!g || !host_out) return fail(FE_EINVAL, "null argument");
    if (!g->ws) return fail(FE_ESTATE, "no workspace bound");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const Geometry& q = g->geo;
    // uses the spectra region as scratch: a running simulation's tensor spectrum (Kt) is untouched
    double* box = reinterpret_cast<double*>(g->ws + g->o_box);
    const int64_t total = (int64_t)q.m[0] * q.m[1] * q.m[2];
    for (int c = 0; c < 6; ++c) {
        FE_CUDA(launch_tensor_box(q, box, c, 1, st));
        FE_CUDA(launch_zero_mode(q, box, c, g->d_eout, st));
        FE_CUDA(cudaMemcpyAsync(host_out + c * total, box, total * sizeof(double), cudaMemcpyDeviceToHost, st));
        FE_CUDA(cudaStreamSynchronize(st));
        g->launches += 2;
    }
    return FE_OK;
}

// ---- a1-a3: electrostatic field of state Y into the E buffer ------------------------------------------
template <typename T>
static fe_status elec_field(fe_grid* g, const T* Y, cudaStream_t st, bool skip_xinv = false)
{
    const Geometry& q = g->geo;
    const int B = g->desc.batch;
    void* S1 = g->ws + g->o_S1;
    void* S2 = g->ws + g->o_S2;
    T* E = reinterpret_cast<T*>(g->ws + g->o_E);
    const T* Kt = reinterpret_cast<const T*>(g->ws + g->o_Kt);
    const int64_t p = q.pitch;
    const int slabs = B * 3 * q.n[2];
    const int64_t rows = (int64_t)slabs * q.n[1];
    const int L = (int)(128 / g->csz), G = q.pitch / L;
    const int nx = q.n[0], ny = q.n[1], nz = q.n[2], My = q.m[1];
    const int Hy = My / 2 + 1, Hz = q.m[2] / 2 + 1;
    const bool tl = g->tiled;
    // strides (complex elements; the tensor table in reals), row-major or tiled (see fe_create_grid)
    const int64_t xspec[4] = {ny, p * ny, tl ? L : p, tl ? (int64_t)ny * L : L};             // S1 as the x passes see it
    const int64_t y1_sa = tl ? L : p, y1_sg = tl ? (int64_t)ny * L : L, y1_sz = p * ny, y1_sb = p * ny * nz;   // S1, y pass
    // tiled S2[b][c][g][z][ky][L]: the y pass reads and writes whole contiguous tiles
    const int64_t y2_sa = tl ? L : p, y2_sg = tl ? (int64_t)My * nz * L : L, y2_sz = tl ? (int64_t)My * L : p * My,
                  y2_sb = p * My * nz;                                                          // S2, y pass
    const int64_t zs[4] = {p * My * nz, tl ? (int64_t)My * L : p * My, tl ? L : p, tl ? (int64_t)My * nz * L : L};
    // bulk-copy y pass (contiguous tiles, ky of S2 in slot order) for the long axes; register-I/O pass otherwise
    const bool use4 = tl && axis4_supported(My);
    int perm[3] = {0, 0, 0};
    if (use4) axis4_radices(My, perm);
    const int64_t ks[4] = {(int64_t)Hz * Hy * p, tl ? L : (int64_t)Hy * p, tl ? (int64_t)Hz * L : p,
                           tl ? (int64_t)Hy * Hz * L : L};
    // x + y passes in one cooperative kernel, S1 planes handed over through a ring that stays in L2 (NEXT-2)
    const bool fuse = use4 && g->opt_fuse_xy && xy_supported(q.m[0] / 2, My, nx, ny);
    // ring: deep enough for every block's X group to run one task ahead of the plane being read (148 blocks / row
    // groups per plane), at least 24 planes, at most 32 MB (it must stay in L2) -- or the caller's FE_OPT_XY_RING
    int ring_slots = g->opt_xy_ring;
    if (ring_slots <= 0) {
        const int rows_task = q.m[0] / 2 >= 256 ? 16 : 32;
        const int64_t plane_bytes = (int64_t)G * ny * 128;
        ring_slots = 3 * (148 * rows_task / ny + 1);
        if (ring_slots < 24) ring_slots = 24;
        while (ring_slots > 8 && ring_slots * plane_bytes > (32ll << 20)) ring_slots /= 2;
    }
    if (ring_slots > slabs) ring_slots = slabs;
    if (ring_slots < 2) ring_slots = 2;
    if (fuse) {
        mark(g, K_XYFWD, st);
        FE_CUDA(launch_xyfwd<T>(g->ctx, Y, S1, S2, nx, ny, nz, slabs, G, ring_slots, y2_sz, y2_sg, y2_sb,
                                reinterpret_cast<int*>(g->ws + g->o_cnt), st));
        g->launches += 2;            // counter reset + kernel
    } else {
    mark(g, K_XFWD, st);
    if (g->fast[0]) FE_CUDA(launch_xfwd2<T>(g->ctx, Y, S1, nx, rows, nx, xspec, L, st));
    else FE_CUDA(launch_xfwd<T>(g->ctx, Y, S1, q.n[0], q.n[1], slabs, q.n[0], (int64_t)q.n[0] * q.n[1], p, p * q.n[1], st));
    mark(g, K_YFWD, st);
    if (g->fast[1]) {
        // tiled: z is the fastest block index, so that concurrently running blocks write neighbouring 128-byte pieces
        if (use4) FE_CUDA(launch_axis4<T>(g->ctx, 1, -1, S1, S2, ny, nz, G, B * 3, y1_sz, y1_sg, y1_sb, y2_sz, y2_sg, y2_sb, st));
        else if (tl) FE_CUDA(launch_axis2<T>(g->ctx, 1, -1, S1, S2, ny, nz, G, B * 3, y1_sa, y1_sz, y1_sg, y1_sb,
                                        y2_sa, y2_sz, y2_sg, y2_sb, st));
        else FE_CUDA(launch_axis2<T>(g->ctx, 1, -1, S1, S2, ny, G, nz, B * 3, y1_sa, y1_sg, y1_sz, y1_sb,
                                     y2_sa, y2_sg, y2_sz, y2_sb, st));
    } else {
        FE_CUDA(launch_axis<T>(g->ctx, 1, -1, S1, S2, q.n[1], q.lanes, q.pitch, q.n[2], B * 3, p, p * q.n[1],
                               p * q.n[1] * q.n[2], p, p * q.m[1], p * q.m[1] * q.n[2], st));
    }
    g->launches += 2;
    }
    mark(g, K_ZMUL, st);
    if (g->fast[2]) FE_CUDA(launch_zmul2<T>(g->ctx, S2, Kt, g->d_members, nz, My, G, B, zs, ks, perm, st));
    else FE_CUDA(launch_zmul<T>(g->ctx, S2, Kt, g->d_members, q.n[2], q.m[1], q.lanes, q.pitch, B, st));
    mark(g, K_YINV, st);
    if (g->fast[1]) {
        if (use4) FE_CUDA(launch_axis4<T>(g->ctx, 1, +1, S2, S1, ny, nz, G, B * 3, y2_sz, y2_sg, y2_sb, y1_sz, y1_sg, y1_sb, st));
        else if (tl) FE_CUDA(launch_axis2<T>(g->ctx, 1, +1, S2, S1, ny, nz, G, B * 3, y2_sa, y2_sz, y2_sg, y2_sb,
                                        y1_sa, y1_sz, y1_sg, y1_sb, st));
        else FE_CUDA(launch_axis2<T>(g->ctx, 1, +1, S2, S1, ny, G, nz, B * 3, y2_sa, y2_sg, y2_sz, y2_sb,
                                     y1_sa, y1_sg, y1_sz, y1_sb, st));
    } else {
        FE_CUDA(launch_axis<T>(g->ctx, 1, +1, S2, S1, q.n[1], q.lanes, q.pitch, q.n[2], B * 3, p, p * q.m[1],
                               p * q.m[1] * q.n[2], p, p * q.n[1], p * q.n[1] * q.n[2], st));
    }
    g->launches += 2;
    if (skip_xinv) return FE_OK;         // the caller runs the x inverse pass slab by slab (FE_OPT_XL_SLABS)
    mark(g, K_XINV, st);
    if (g->fast[0]) FE_CUDA(launch_xinv2<T>(g->ctx, S1, E, nx, rows, nx, xspec, L, st));
    else FE_CUDA(launch_xinv<T>(g->ctx, S1, E, q.n[0], q.n[1], slabs, p, p * q.n[1], q.n[0], (int64_t)q.n[0] * q.n[1], st));
    g->launches += 1;
    return FE_OK;
}

// folded stage combination of the multistep / embedded integrators (LocalArgs::kOut, lk, lc)
struct StageLin {
    void* kOut = nullptr;
    const void* lk[4] = {nullptr, nullptr, nullptr, nullptr};
    double lc[4] = {0, 0, 0, 0};
    int nlin = 0;
    void add(const void* k, double c) { if (c != 0.0) { lk[nlin] = k; lc[nlin] = c; ++nlin; } }
};

template <typename T>
static fe_status stage(fe_grid* g, const T* Y, const T* baseY, T* Yout, double cy, const T* accIn, T* accOut, double ca,
                       uint32_t terms, cudaStream_t st, const StageLin* lin = nullptr)
{
    const bool elec = (terms & FE_TERM_ELEC) != 0;
    // FE_OPT_XL_SLABS > 1: E_elec goes from the x inverse pass to the local step slab by slab through the first
    // planes of each component's region of the E buffer, which every slab overwrites and which so stay in L2 (no round trip through HBM)
    const Geometry& q = g->geo;
    const int Lx = (int)(128 / g->csz);
    const int nslab = elec && g->opt_xl_slabs > 1 && g->fast[0] && g->tiled && q.n[2] >= g->opt_xl_slabs &&
                              xinv_slab_supported(q.m[0] / 2, q.n[0], q.n[1], Lx, sizeof(T))
                          ? g->opt_xl_slabs
                          : 1;
    if (elec) {
        fe_status s = elec_field<T>(g, Y, st, nslab > 1);
        if (s != FE_OK) return s;
    }
    LocalArgs a;
    memset(&a, 0, sizeof(a));
    a.Y = Y;
    a.Eelec = elec ? g->ws + g->o_E : nullptr;
    a.baseY = baseY;
    a.Yout = Yout;
    a.accIn = accIn;
    a.accOut = accOut;
    a.cy = cy;
    a.ca = ca;
    if (lin) {
        a.kOut = lin->kOut;
        a.nlin = lin->nlin;
        for (int j = 0; j < lin->nlin; ++j) { a.lk[j] = lin->lk[j]; a.lc[j] = lin->lc[j]; }
    }
    a.map = g->map;
    a.mats = g->d_mats;
    a.members = g->d_members;
    a.nmat = g->desc.n_materials;
    for (int i = 0; i < 3; ++i) { a.n[i] = g->geo.n[i]; a.periodic[i] = g->geo.periodic[i]; a.d[i] = g->geo.d[i]; }
    a.terms = terms;
    a.batch = g->desc.batch;
    a.mixed = g->mixed;
    a.vac0 = g->vac0;
    a.t = g->tstage;
    if (nslab > 1) {
        const int64_t p = q.pitch;
        const int nx = q.n[0], ny = q.n[1], nz = q.n[2];
        const int64_t xspec[4] = {ny, p * ny, Lx, (int64_t)ny * Lx};      // tiled S1 as the x passes see it
        for (int k = 0; k < nslab; ++k) {
            const int zb = (int)((int64_t)nz * k / nslab), ze = (int)((int64_t)nz * (k + 1) / nslab);
            mark(g, K_XINV, st);
            FE_CUDA(launch_xinv2_slab<T>(g->ctx, g->ws + g->o_S1, reinterpret_cast<T*>(g->ws + g->o_E), nx, g->desc.batch * 3, ny,
                                         nz, zb, ze - zb, xspec, Lx, st));
            a.zbeg = zb;
            a.zend = ze;
            a.e_z0 = zb;
            mark(g, K_LOCAL, st);
            FE_CUDA(launch_local<T>(a, st));
            g->launches += 2;
        }
        return FE_OK;
    }
    mark(g, K_LOCAL, st);
    FE_CUDA(launch_local<T>(a, st));
    g->launches += 1;
    return FE_OK;
}

static fe_status check_ready(fe_grid* g, const void* P, uint32_t terms)
{
    if (!g || !P) return fail(FE_EINVAL, "null argument");
    if (terms & ~(uint32_t)FE_TERM_ALL) return fail(FE_EINVAL, "unknown bits in terms");
    if (reinterpret_cast<uintptr_t>(P) % 16) return fail(FE_EINVAL, "state arrays must be 16-byte aligned");
    if (!g->ws) return fail(FE_ESTATE, "no workspace bound");
    if ((terms & FE_TERM_ELEC) && !g->tensor_ready)
        return fail(FE_ESTATE, "FE_TERM_ELEC requested before fe_precompute_tensor");
    return FE_OK;
}

extern "C" fe_status fe_rhs(fe_grid* g, const void* P, void* dPdt, uint32_t terms, void* stream)
{
    fe_status s = check_ready(g, P, terms);
    if (s != FE_OK) return s;
    if (!dPdt || dPdt == P) return fail(FE_EINVAL, "dPdt must be a distinct array");
    if (reinterpret_cast<uintptr_t>(dPdt) % 16) return fail(FE_EINVAL, "state arrays must be 16-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if ((s = sync_params(g, st)) != FE_OK) return s;
    g->tstage = g->time;
    s = g->f32 ? stage<float>(g, (const float*)P, nullptr, (float*)dPdt, 1.0, nullptr, nullptr, 0.0, terms, st)
               : stage<double>(g, (const double*)P, nullptr, (double*)dPdt, 1.0, nullptr, nullptr, 0.0, terms, st);
    mark(g, -1, st);
    return s;
}

template <typename T>
static fe_status step_T(fe_grid* g, T* P, double dt, int nsteps, int integ, uint32_t terms, cudaStream_t st, double t0)
{
    T* Y = reinterpret_cast<T*>(g->ws + g->o_Y);
    T* ACC = reinterpret_cast<T*>(g->ws + g->o_ACC);
    T* PP = reinterpret_cast<T*>(g->ws + g->o_PP);
    const size_t bytes = (size_t)g->desc.batch * 3 * g->N * sizeof(T);
    fe_status s;
    if (integ == FE_EULER) {
        T* cur = P;
        T* nxt = PP;
        for (int i = 0; i < nsteps; ++i) {
            g->tstage = t0 + i * dt;
            if ((s = stage<T>(g, cur, cur, nxt, dt, nullptr, nullptr, 0.0, terms, st)) != FE_OK) return s;
            T* t = cur; cur = nxt; nxt = t;
        }
        if (cur != P) {
            mark(g, K_OTHER, st);
            FE_CUDA(cudaMemcpyAsync(P, cur, bytes, cudaMemcpyDeviceToDevice, st));
        }
    } else if (integ == FE_HEUN) {
        for (int i = 0; i < nsteps; ++i) {
            // k1 = f(P): Y = P + dt k1, ACC = P + dt/2 k1;  k2 = f(Y): P = ACC + dt/2 k2
            const double tn = t0 + i * dt;
            g->tstage = tn;
            if ((s = stage<T>(g, P, P, Y, dt, P, ACC, 0.5 * dt, terms, st)) != FE_OK) return s;
            g->tstage = tn + dt;
            if ((s = stage<T>(g, Y, ACC, P, 0.5 * dt, nullptr, nullptr, 0.0, terms, st)) != FE_OK) return s;
        }
    } else if (integ == FE_AB3M2) {
        // P* = P + dt/12 (23 f_n - 16 f_{n-1} + 5 f_{n-2}) (Euler predictor while there is no history),
        // P <- P + dt/2 (f_n + f(P*)); the history restarts with every call
        T* F[3] = {reinterpret_cast<T*>(g->ws + g->o_K[0]), reinterpret_cast<T*>(g->ws + g->o_K[1]),
                   reinterpret_cast<T*>(g->ws + g->o_K[2])};
        for (int i = 0; i < nsteps; ++i) {
            // both stage combinations ride on the local step's epilogue (no separate streaming passes):
            //   f_n = f(P) -> F[0],  P* = P + [c1 f_{n-1} + c2 f_{n-2}] + c0 f_n -> Y;   P <- P + dt/2 f_n + dt/2 f(P*)
            const double tn = t0 + i * dt;
            g->tstage = tn;
            StageLin pre;
            pre.kOut = F[0];
            double c0 = dt;
            if (i >= 2) {
                c0 = dt * 23.0 / 12.0;
                pre.add(F[1], -dt * 16.0 / 12.0);
                pre.add(F[2], dt * 5.0 / 12.0);
            }
            if ((s = stage<T>(g, P, P, Y, c0, nullptr, nullptr, 0.0, terms, st, &pre)) != FE_OK) return s;
            g->tstage = tn + dt;
            StageLin cor;
            cor.add(F[0], 0.5 * dt);
            if ((s = stage<T>(g, Y, P, P, 0.5 * dt, nullptr, nullptr, 0.0, terms, st, &cor)) != FE_OK) return s;
            T* t = F[2]; F[2] = F[1]; F[1] = F[0]; F[0] = t;
        }
    } else {
        for (int i = 0; i < nsteps; ++i) {
            // classical RK4, weights 1/6 1/3 1/3 1/6, stage points P + dt/2 k1, P + dt/2 k2, P + dt k3
            const double tn = t0 + i * dt;
            g->tstage = tn;
            if ((s = stage<T>(g, P, P, Y, 0.5 * dt, P, ACC, dt / 6.0, terms, st)) != FE_OK) return s;
            g->tstage = tn + dt / 2.0;
            if ((s = stage<T>(g, Y, P, PP, 0.5 * dt, ACC, ACC, dt / 3.0, terms, st)) != FE_OK) return s;
            if ((s = stage<T>(g, PP, P, Y, dt, ACC, ACC, dt / 3.0, terms, st)) != FE_OK) return s;
            g->tstage = tn + dt;
            if ((s = stage<T>(g, Y, ACC, P, dt / 6.0, nullptr, nullptr, 0.0, terms, st)) != FE_OK) return s;
        }
    }
    return FE_OK;
}

extern "C" fe_status fe_step(fe_grid* g, void* P, double dt, int32_t nsteps, int32_t integ, uint32_t terms, void* stream)
{
    fe_status s = check_ready(g, P, terms);
    if (s != FE_OK) return s;
    if (nsteps < 0) return fail(FE_EINVAL, "nsteps < 0");
    if (!isfinite(dt)) return fail(FE_EINVAL, "dt not finite");
    if (integ != FE_EULER && integ != FE_HEUN && integ != FE_RK4 && integ != FE_AB3M2) return fail(FE_EINVAL, "unknown integrator");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if ((s = sync_params(g, st)) != FE_OK) return s;
    const double time0 = g->time;
    auto run = [&](int n, cudaStream_t on) {
        return g->f32 ? step_T<float>(g, (float*)P, dt, n, integ, terms, on, time0)
                      : step_T<double>(g, (double*)P, dt, n, integ, terms, on, time0);
    };
    // Long runs replay a CUDA graph of one unit of steps (2 Euler steps: the ping-pong returns to P; 1 Heun / RK4 step)
    // on an internal stream ordered with the caller's stream by events: small grids are launch bound otherwise.
    // The first unit always runs eagerly (one-time kernel attribute set-up must not happen inside a capture).
    const int unit = integ == FE_EULER ? 2 : 1;
    if (g->prof_on || g->goff || nsteps < 6 * unit || integ == FE_AB3M2 || g->any_wave) {
        s = run(nsteps, st);             // (a time-dependent E_ext changes the kernel arguments from step to step)
        if (s == FE_OK) g->time = time0 + nsteps * dt;
        mark(g, -1, st);
        return s;
    }
    if ((s = run(unit, st)) != FE_OK) return s;
    int left = nsteps - unit;
    const int reps = left / unit;
    bool ok = true;
    if (!g->gstream) {
        ok = cudaStreamCreateWithFlags(&g->gstream, cudaStreamNonBlocking) == cudaSuccess &&
             cudaEventCreateWithFlags(&g->gev_in, cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&g->gev_out, cudaEventDisableTiming) == cudaSuccess;
    }
    if (ok && !(g->gvalid && g->gP == P && g->gdt == dt && g->ginteg == integ && g->gterms == terms)) {
        if (g->gexec) { cudaGraphExecDestroy(g->gexec); g->gexec = nullptr; }
        g->gvalid = false;
        cudaGraph_t graph = nullptr;
        const uint64_t l0 = g->launches;
        ok = cudaStreamBeginCapture(g->gstream, cudaStreamCaptureModeRelaxed) == cudaSuccess;
        if (ok) {
            const fe_status cs = run(unit, g->gstream);
            const cudaError_t ce = cudaStreamEndCapture(g->gstream, &graph);
            ok = cs == FE_OK && ce == cudaSuccess && graph != nullptr;
        }
        g->gunit_launches = g->launches - l0;
        g->launches = l0;                                   // the captured unit did not run
        if (ok) ok = cudaGraphInstantiate(&g->gexec, graph, 0) == cudaSuccess;
        if (graph) cudaGraphDestroy(graph);
        if (ok) { g->gvalid = true; g->gP = P; g->gdt = dt; g->ginteg = integ; g->gterms = terms; }
    }
    if (ok) {
        ok = cudaEventRecord(g->gev_in, st) == cudaSuccess && cudaStreamWaitEvent(g->gstream, g->gev_in, 0) == cudaSuccess;
        for (int r = 0; ok && r < reps; ++r) ok = cudaGraphLaunch(g->gexec, g->gstream) == cudaSuccess;
        if (ok) ok = cudaEventRecord(g->gev_out, g->gstream) == cudaSuccess && cudaStreamWaitEvent(st, g->gev_out, 0) == cudaSuccess;
        if (ok) {
            g->launches += (uint64_t)reps * g->gunit_launches;
            left -= reps * unit;
        } else {
            return fail(FE_ECUDA, "CUDA graph replay failed: %s", cudaGetErrorString(cudaGetLastError()));
        }
    } else {
        cudaGetLastError();                                 // capture unavailable: run eagerly from now on
        g->goff = true;
        g->gvalid = false;
    }
    s = left > 0 ? run(left, st) : FE_OK;
    if (s == FE_OK) g->time = time0 + nsteps * dt;
    mark(g, -1, st);
    return s;
}

// ---- adaptive Cash-Karp RK45 (include/fe.h states the controller) ----------------
template <typename T>
static fe_status rk45_T(fe_grid* g, T* P, double t_span, double dt_init, double tol, int max_steps, uint32_t terms,
                        fe_rk45_stats* out, cudaStream_t st)
{
    static const double A[6][5] = {{0, 0, 0, 0, 0},
                                   {1.0 / 5.0, 0, 0, 0, 0},
                                   {3.0 / 40.0, 9.0 / 40.0, 0, 0, 0},
                                   {3.0 / 10.0, -9.0 / 10.0, 6.0 / 5.0, 0, 0},
                                   {-11.0 / 54.0, 5.0 / 2.0, -70.0 / 27.0, 35.0 / 27.0, 0},
                                   {1631.0 / 55296.0, 175.0 / 512.0, 575.0 / 13824.0, 44275.0 / 110592.0, 253.0 / 4096.0}};
    static const double C[6] = {0.0, 1.0 / 5.0, 3.0 / 10.0, 3.0 / 5.0, 1.0, 7.0 / 8.0};
    static const double B5[6] = {37.0 / 378.0, 0.0, 250.0 / 621.0, 125.0 / 594.0, 0.0, 512.0 / 1771.0};
    static const double B4[6] = {2825.0 / 27648.0, 0.0, 18575.0 / 48384.0, 13525.0 / 55296.0, 277.0 / 14336.0, 1.0 / 4.0};
    T* K[6];
    for (int j = 0; j < 6; ++j) K[j] = reinterpret_cast<T*>(g->ws + g->o_K[j]);
    T* Y = reinterpret_cast<T*>(g->ws + g->o_Y);
    T* Y5 = reinterpret_cast<T*>(g->ws + g->o_PP);
    const int64_t n = (int64_t)g->desc.batch * 3 * g->N;
    const size_t bytes = (size_t)n * sizeof(T);
    const double time0 = g->time;
    double t = 0.0, dt = dt_init, err = 0.0, dt_last = 0.0;
    int acc = 0, rej = 0, evals = 0, nonfinite = 0;
    fe_status s;
    while (t < t_span && acc + rej < max_steps) {
        const double h = dt < t_span - t ? dt : t_span - t;
        // stage i evaluates K[i] = f(Y_i) and, in the same epilogue, forms Y_{i+1} = P + h sum_{j <= i} a_{i+1,j} K[j]
        // (terms in ascending j, the stage's own k last); the stage states alternate between two buffers
        T* Yab[2] = {Y, reinterpret_cast<T*>(g->ws + g->o_ACC)};
        for (int i = 0; i < 6; ++i) {
            const T* Yi = i == 0 ? P : Yab[(i - 1) & 1];
            g->tstage = time0 + t + C[i] * h;
            if (i < 5) {
                StageLin lin;
                lin.kOut = K[i];
                for (int j = 0; j < i; ++j) lin.add(K[j], h * A[i + 1][j]);
                if ((s = stage<T>(g, Yi, P, Yab[i & 1], h * A[i + 1][i], nullptr, nullptr, 0.0, terms, st, &lin)) != FE_OK) return s;
            } else {
                if ((s = stage<T>(g, Yi, nullptr, K[i], 1.0, nullptr, nullptr, 0.0, terms, st)) != FE_OK) return s;
            }
        }
        evals += 6;
        LinArgs b5, d;
        for (int j = 0; j < 6; ++j) { b5.k[j] = d.k[j] = K[j]; b5.c[j] = h * B5[j]; d.c[j] = h * (B5[j] - B4[j]); }
        FE_CUDA(launch_rk45_final<T>(Y5, P, b5, d, n, g->d_eout, st));
        g->launches += 1;
        double emax = 0.0;
        FE_CUDA(cudaMemcpyAsync(&emax, g->d_eout, sizeof(double), cudaMemcpyDeviceToHost, st));
        FE_CUDA(cudaStreamSynchronize(st));
        err = emax / tol;
        if (err <= 1.0) {                                // NaN compares false: a non-finite estimate rejects
            FE_CUDA(cudaMemcpyAsync(P, Y5, bytes, cudaMemcpyDeviceToDevice, st));
            t += h; ++acc; dt_last = h; nonfinite = 0;
            dt = err <= 1.89e-4 ? 5.0 * h : 0.9 * h * pow(err, -0.2);
        } else {
            ++rej;
            const double shr = 0.9 * h * pow(err, -0.25);
            dt = (shr > 0.1 * h) ? shr : 0.1 * h;         // also taken when err is NaN
            // a stage that overflowed may recover with a smaller step; a state that already holds NaN / Inf never does
            if (isfinite(err)) nonfinite = 0;
            else if (++nonfinite >= 8) {
                g->time = time0 + t;
                if (out) { out->t = t; out->dt_last = dt_last; out->dt_next = dt; out->err_last = err;
                           out->accepted = acc; out->rejected = rej; out->rhs_evals = evals; }
                return fail(FE_ENONFINITE, "RK45: non-finite error estimate in 8 consecutive attempts");
            }
        }
    }
    FE_CUDA(cudaStreamSynchronize(st));
    g->time = time0 + t;
    if (out) { out->t = t; out->dt_last = dt_last; out->dt_next = dt; out->err_last = err;
               out->accepted = acc; out->rejected = rej; out->rhs_evals = evals; }
    return FE_OK;
}

extern "C" fe_status fe_step_rk45(fe_grid* g, void* P, double t_span, double dt_init, double tol, int32_t max_steps,
                                  uint32_t terms, fe_rk45_stats* stats, void* stream)
{
    fe_status s = check_ready(g, P, terms);
    if (s != FE_OK) return s;
    if (!(t_span >= 0.0) || !(dt_init > 0.0) || !(tol > 0.0) || !isfinite(t_span) || !isfinite(dt_init) || max_steps < 0)
        return fail(FE_EINVAL, "RK45: t_span >= 0, dt_init > 0, tol > 0, max_steps >= 0 required");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if ((s = sync_params(g, st)) != FE_OK) return s;
    s = g->f32 ? rk45_T<float>(g, (float*)P, t_span, dt_init, tol, max_steps, terms, stats, st)
               : rk45_T<double>(g, (double*)P, t_span, dt_init, tol, max_steps, terms, stats, st);
    mark(g, -1, st);
    return s;
}

extern "C" fe_status fe_energy(fe_grid* g, const void* P, uint32_t terms, double* host_out, void* stream)
{
    fe_status s = check_ready(g, P, terms);
    if (s != FE_OK) return s;
    if (!host_out) return fail(FE_EINVAL, "null argument");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if ((s = sync_params(g, st)) != FE_OK) return s;
    const bool elec = (terms & FE_TERM_ELEC) != 0;
    if (elec) {
        s = g->f32 ? elec_field<float>(g, (const float*)P, st) : elec_field<double>(g, (const double*)P, st);
        if (s != FE_OK) return s;
    }
    EnergyArgs a;
    memset(&a, 0, sizeof(a));
    a.P = P;
    a.Eelec = elec ? g->ws + g->o_E : nullptr;
    a.map = g->map;
    a.mats = g->d_mats;
    a.members = g->d_members;
    a.nmat = g->desc.n_materials;
    for (int i = 0; i < 3; ++i) { a.n[i] = g->geo.n[i]; a.periodic[i] = g->geo.periodic[i]; a.d[i] = g->geo.d[i]; }
    a.terms = terms;
    a.batch = g->desc.batch;
    a.partials = reinterpret_cast<double*>(g->ws + g->o_part);
    a.out = g->d_eout;
    a.nblk = g->nblk;
    a.t = g->time;
    FE_CUDA(g->f32 ? launch_energy<float>(a, st) : launch_energy<double>(a, st));
    g->launches += 2;
    const size_t nb = (size_t)g->desc.batch * 8;
    FE_CUDA(cudaMemcpyAsync(host_out, g->d_eout, nb * sizeof(double), cudaMemcpyDeviceToHost, st));
    FE_CUDA(cudaStreamSynchronize(st));
    for (size_t i = 0; i < nb; ++i)
        if (!isfinite(host_out[i])) return fail(FE_ENONFINITE, "non-finite energy or mean (entry %zu)", i);
    return FE_OK;
}

// ---- a6 without any allocation: partial sums in a static device array ---------------------------------
// Scratch of fe_energy_noalloc: [B][nblk][8] partial sums of k_energy.  File-scope device memory: every GPU that loads the
// library holds these 512 KiB until the process exits.  In host code the NAME of the array is a host-side stand-in, not a
// device address; the address a kernel may use comes from cudaGetSymbolAddress, once per device with that device current.
constexpr size_t kNoAllocDoubles = 65536;                               // 512 KiB: batch * 296 blocks * 8 sums, batch <= 27
static __device__ __align__(256) double g_noalloc_partials[kNoAllocDoubles];

extern "C" fe_status fe_energy_noalloc(fe_grid* g, const void* P, uint32_t terms, double* dev_out, void* stream)
{
    fe_status s = check_ready(g, P, terms);
    if (s != FE_OK) return s;
    if (!dev_out) return fail(FE_EINVAL, "null argument");
    const size_t need = (size_t)g->desc.batch * g->nblk * 8;
    if (need > kNoAllocDoubles)
        return fail(FE_EINVAL, "fe_energy_noalloc: batch %d needs %zu partial sums, the static scratch holds %zu (batch <= %zu)",
                    g->desc.batch, need, kNoAllocDoubles, kNoAllocDoubles / ((size_t)g->nblk * 8));
    static PerDevice<double*> cache;                                    // device address of the array, per device
    double*& scratch = cache.here();
    if (!scratch) {
        double* ptr = nullptr;
        FE_CUDA(cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_noalloc_partials));
        if (!ptr) return fail(FE_ECUDA, "cudaGetSymbolAddress returned a null address");
        scratch = ptr;
    }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if ((s = sync_params(g, st)) != FE_OK) return s;
    const bool elec = (terms & FE_TERM_ELEC) != 0;
    if (elec) {
        s = g->f32 ? elec_field<float>(g, (const float*)P, st) : elec_field<double>(g, (const double*)P, st);
        if (s != FE_OK) return s;
    }
    EnergyArgs a;
    memset(&a, 0, sizeof(a));
    a.P = P;
    a.Eelec = elec ? g->ws + g->o_E : nullptr;
    a.map = g->map;
    a.mats = g->d_mats;
    a.members = g->d_members;
    a.nmat = g->desc.n_materials;
    for (int i = 0; i < 3; ++i) { a.n[i] = g->geo.n[i]; a.periodic[i] = g->geo.periodic[i]; a.d[i] = g->geo.d[i]; }
    a.terms = terms;
    a.batch = g->desc.batch;
    a.partials = scratch;             // every row [b][block][0..7] is written by its block before it is summed: nothing to clear
    a.out = dev_out;
    a.nblk = g->nblk;
    a.t = g->time;
    FE_CUDA(g->f32 ? launch_energy<float>(a, st) : launch_energy<double>(a, st));
    g->launches += 2;
    return FE_OK;
}

// ---- per-kernel timing (bench.py's roofline leg) ------------------------------------------------------
extern "C" fe_status fe_profile(fe_grid* g, int32_t enable)
{
    if (!g) return fail(FE_EINVAL, "null argument");
    g->prof_on = enable != 0;
    g->prof_used = 0;
    return FE_OK;
}

extern "C" fe_status fe_profile_read(fe_grid* g, double* host_ms, uint64_t* host_counts, void* stream)
{
    if (!g || !host_ms || !host_counts) return fail(FE_EINVAL, "null argument");
    FE_CUDA(cudaStreamSynchronize(static_cast<cudaStream_t>(stream)));
    for (int k = 0; k < K_NKINDS; ++k) { host_ms[k] = 0.0; host_counts[k] = 0; }
    for (size_t i = 0; i + 1 < g->prof_used; ++i) {
        const int kind = g->prof_kind[i];
        if (kind < 0) continue;
        float ms = 0.f;
        FE_CUDA(cudaEventElapsedTime(&ms, g->prof_ev[i], g->prof_ev[i + 1]));
        host_ms[kind] += ms;
        host_counts[kind] += 1;
    }
    g->prof_used = 0;
    return FE_OK;
}
