/* fe_oracle.c -- plain, slow CPU oracle for the TDGL hot path of arxiv/paper_2605_28800.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference leg may load this library.  It shares no source, header,
 * table or constant with the CUDA path (paper_2605_28800_b200/csrc) and neither imports the other.
 *
 * What it computes (one simulation; batches are looped over by the caller):
 *   O1  Landau energy density and its derivative          PAPER.md:41-47 (Eq. 3), 211 (per-axis a1)
 *   O2  discrete gradient energy and its exact derivative PAPER.md:53-58 (Eq. 4), reading A2
 *   O3  cell-averaged dipolar tensor (__float128) and the direct O(N^2) electrostatic sum
 *                                                         PAPER.md:66-76 (Eq. 5-6), readings A3, A4
 * Everything is the plain definition: no blocking, no FFT, no symmetry tricks in the field sum.
 * The only concession to run time is that the tensor table evaluates the Newell primitives once
 * per lattice point (they are shared by the 27 terms of neighbouring entries) and that loops
 * over independent outputs carry "#pragma omp parallel for".
 *
 * Layout: fields are [3][nz][ny][nx] doubles (x fastest); material map [nz][ny][nx] bytes.
 * Pins: tests/test_oracle_*.py.  No function here is unpinned.
 */
#include <math.h>
#include <quadmath.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef __float128 q_t;

typedef struct {
    double a1[3];
    double a11, a12, a111, a112, a123;
    double a1111, a1112, a1122, a1123;
    int32_t active;
} orc_landau;

/* ------------------------------------------------------------------------------------------
 * O1. Landau (Eq. 3 + 8th-order cubic-symmetry slots, zero for the paper's Table 1).
 * With a = Px^2, b = Py^2, c = Pz^2.
 * ---------------------------------------------------------------------------------------- */
double orc_landau_f(const orc_landau* m, const double* P)
{
    double a = P[0] * P[0], b = P[1] * P[1], c = P[2] * P[2];
    double f = m->a1[0] * a + m->a1[1] * b + m->a1[2] * c;
    f += m->a11 * (a * a + b * b + c * c);
    f += m->a12 * (a * b + b * c + c * a);
    f += m->a111 * (a * a * a + b * b * b + c * c * c);
    f += m->a112 * (a * a * (b + c) + b * b * (a + c) + c * c * (a + b));
    f += m->a123 * a * b * c;
    f += m->a1111 * (a * a * a * a + b * b * b * b + c * c * c * c);
    f += m->a1112 * (a * a * a * (b + c) + b * b * b * (a + c) + c * c * c * (a + b));
    f += m->a1122 * (a * a * b * b + b * b * c * c + c * c * a * a);
    f += m->a1123 * a * b * c * (a + b + c);
    return f;
}

/* d f / d P_i for i = 0 with (a1i, Pi, a, b, c) = own axis first, the other two after it. */
static double dfd_one(const orc_landau* m, double a1i, double Pi, double a, double b, double c)
{
    double s = 2.0 * a1i + 4.0 * m->a11 * a + 2.0 * m->a12 * (b + c) + 6.0 * m->a111 * a * a;
    s += m->a112 * (4.0 * a * (b + c) + 2.0 * (b * b + c * c));
    s += 2.0 * m->a123 * b * c;
    s += 8.0 * m->a1111 * a * a * a;
    s += m->a1112 * (6.0 * a * a * (b + c) + 2.0 * (b * b * b + c * c * c));
    s += 4.0 * m->a1122 * a * (b * b + c * c);
    s += m->a1123 * (4.0 * a * b * c + 2.0 * b * c * (b + c));
    return Pi * s;
}

void orc_landau_dfdp(const orc_landau* m, const double* P, double* out)
{
    double a = P[0] * P[0], b = P[1] * P[1], c = P[2] * P[2];
    out[0] = dfd_one(m, m->a1[0], P[0], a, b, c);
    out[1] = dfd_one(m, m->a1[1], P[1], b, c, a);
    out[2] = dfd_one(m, m->a1[2], P[2], c, a, b);
}

/* Landau field E_Land = -df/dP on the grid (0 in vacuum cells) and energy density sum. */
void orc_landau_field(const orc_landau* mats, const uint8_t* matmap, int64_t N,
                      const double* P, double* E)
{
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < N; ++r) {
        const orc_landau* m = &mats[matmap ? matmap[r] : 0];
        double p[3] = { P[r], P[N + r], P[2 * N + r] }, d[3] = { 0, 0, 0 };
        if (m->active) orc_landau_dfdp(m, p, d);
        E[r] = -d[0]; E[N + r] = -d[1]; E[2 * N + r] = -d[2];
    }
}

double orc_landau_energy_sum(const orc_landau* mats, const uint8_t* matmap, int64_t N, const double* P)
{
    long double s = 0;
    for (int64_t r = 0; r < N; ++r) {
        const orc_landau* m = &mats[matmap ? matmap[r] : 0];
        double p[3] = { P[r], P[N + r], P[2 * N + r] };
        if (m->active) s += orc_landau_f(m, p);
    }
    return (double)s;       /* caller multiplies by the cell volume V */
}

/* ------------------------------------------------------------------------------------------
 * O2. Gradient energy (Eq. 4), discrete reading A2.
 *   c_ia = G11 if a == i else (G44 + G44')            Gm = G12 + G44 - G44'
 *   F_h/V = sum_r { sum_i sum_a 1/2 c_ia [(P_i(r+e_a) - P_i(r))/D_a]^2   (bond: both cells active)
 *                 + Gm sum_{i<j} (D_i P_i)(r) (D_j P_j)(r) }
 *   (D_a u)(r) = (u(r+e_a) - u(r-e_a)) / (2 D_a), u = 0 outside the grid and in vacuum cells
 *   (open axis) or wrapped (periodic axis); the r-sum of the mixed term runs over every grid cell.
 *   E_i(r) = -(1/V) dF_h/dP_i(r).
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    int n[3];               /* nx, ny, nz */
    double d[3];
    int periodic[3];
    const uint8_t* act;     /* [nz][ny][nx] 1 = active cell */
    const double* P;        /* [3][N] */
} grid_view;

/* value of component i at integer cell (x,y,z) shifted by s; 0 if outside (open) or vacuum;
 * *exists tells whether that cell is an active in-grid cell. */
static double cell_val(const grid_view* g, int i, int x, int y, int z, int* exists)
{
    int c[3] = { x, y, z };
    for (int a = 0; a < 3; ++a) {
        if (c[a] < 0 || c[a] >= g->n[a]) {
            if (!g->periodic[a]) { if (exists) *exists = 0; return 0.0; }
            c[a] = ((c[a] % g->n[a]) + g->n[a]) % g->n[a];
        }
    }
    int64_t N = (int64_t)g->n[0] * g->n[1] * g->n[2];
    int64_t r = ((int64_t)c[2] * g->n[1] + c[1]) * g->n[0] + c[0];
    if (!g->act[r]) { if (exists) *exists = 0; return 0.0; }
    if (exists) *exists = 1;
    return g->P[(int64_t)i * N + r];
}

static double central_diff(const grid_view* g, int i, int a, int x, int y, int z)
{
    int e[3] = { 0, 0, 0 };
    e[a] = 1;
    double up = cell_val(g, i, x + e[0], y + e[1], z + e[2], NULL);
    double dn = cell_val(g, i, x - e[0], y - e[1], z - e[2], NULL);
    return (up - dn) / (2.0 * g->d[a]);
}

double orc_grad_energy_sum(const int* n, const double* d, const int* periodic, const uint8_t* act,
                           const double* P, double G11, double G12, double G44, double G44p)
{
    grid_view g = { { n[0], n[1], n[2] }, { d[0], d[1], d[2] },
                    { periodic[0], periodic[1], periodic[2] }, act, P };
    double Gm = G12 + G44 - G44p;
    long double s = 0;
    for (int z = 0; z < n[2]; ++z)
        for (int y = 0; y < n[1]; ++y)
            for (int x = 0; x < n[0]; ++x) {
                int here;
                (void)cell_val(&g, 0, x, y, z, &here);
                for (int i = 0; i < 3; ++i)
                    for (int a = 0; a < 3; ++a) {
                        /* forward bond r -> r + e_a, counted once; on a periodic axis the last
                         * cell bonds to the first. */
                        int e[3] = { 0, 0, 0 };
                        e[a] = 1;
                        int there;
                        double pu = cell_val(&g, i, x + e[0], y + e[1], z + e[2], &there);
                        if (!here || !there) continue;
                        double p0 = cell_val(&g, i, x, y, z, NULL);
                        double cia = (a == i) ? G11 : (G44 + G44p);
                        double q = (pu - p0) / d[a];
                        s += 0.5 * cia * q * q;
                    }
                double D0 = central_diff(&g, 0, 0, x, y, z);
                double D1 = central_diff(&g, 1, 1, x, y, z);
                double D2 = central_diff(&g, 2, 2, x, y, z);
                s += Gm * (D0 * D1 + D1 * D2 + D2 * D0);
            }
    return (double)s;       /* caller multiplies by V */
}

void orc_grad_field(const int* n, const double* d, const int* periodic, const uint8_t* act,
                    const double* P, double G11, double G12, double G44, double G44p, double* E)
{
    grid_view g = { { n[0], n[1], n[2] }, { d[0], d[1], d[2] },
                    { periodic[0], periodic[1], periodic[2] }, act, P };
    double Gm = G12 + G44 - G44p;
    int64_t N = (int64_t)n[0] * n[1] * n[2];
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < n[2]; ++z)
        for (int y = 0; y < n[1]; ++y)
            for (int x = 0; x < n[0]; ++x) {
                int64_t r = ((int64_t)z * n[1] + y) * n[0] + x;
                int c[3] = { x, y, z };
                for (int i = 0; i < 3; ++i) {
                    double acc = 0.0;
                    if (act[r]) {
                        double p0 = P[(int64_t)i * N + r];
                        for (int a = 0; a < 3; ++a) {
                            int e[3] = { 0, 0, 0 };
                            e[a] = 1;
                            double cia = (a == i) ? G11 : (G44 + G44p);
                            int ex;
                            double pu = cell_val(&g, i, x + e[0], y + e[1], z + e[2], &ex);
                            if (ex) acc += cia * (pu - p0) / (d[a] * d[a]);   /* missing bond: 0 */
                            double pd = cell_val(&g, i, x - e[0], y - e[1], z - e[2], &ex);
                            if (ex) acc += cia * (pd - p0) / (d[a] * d[a]);
                        }
                        for (int j = 0; j < 3; ++j) {
                            if (j == i) continue;
                            /* Gm * (D_i D_j P_j)(r); D_i is the grid-truncated operator: the
                             * intermediate cell r +- e_i must be inside the grid (or wrap). */
                            double t = 0.0;
                            for (int si = -1; si <= 1; si += 2) {
                                int ci = c[i] + si;
                                if ((ci < 0 || ci >= n[i]) && !periodic[i]) continue;
                                int q[3] = { x, y, z };
                                q[i] += si;
                                t += si * central_diff(&g, j, j, q[0], q[1], q[2]);
                            }
                            acc += Gm * t / (2.0 * d[i]);
                        }
                    }
                    E[(int64_t)i * N + r] = acc;
                }
            }
}

/* ------------------------------------------------------------------------------------------
 * O3. Cell-averaged dipolar tensor, Newell-Williams-Dunlop closed form in __float128.
 *   N_ij(R) = -(1/(4 pi V)) int_cell d3r int_cell d3r' d_i d_j (1/|R + r - r'|)
 *   4 pi V N_xx = -d2x d2y d2z f,  4 pi V N_xy = -d2x d2y d2z g   (second differences, step D_a)
 * ---------------------------------------------------------------------------------------- */
static q_t newell_f(q_t x, q_t y, q_t z)
{
    x = fabsq(x); y = fabsq(y); z = fabsq(z);                 /* f is even in x, y, z */
    q_t x2 = x * x, y2 = y * y, z2 = z * z, R = sqrtq(x2 + y2 + z2), r = 0;
    if (y != 0 && x2 + z2 != 0) r += (y / 2) * (z2 - x2) * asinhq(y / sqrtq(x2 + z2));
    if (z != 0 && x2 + y2 != 0) r += (z / 2) * (y2 - x2) * asinhq(z / sqrtq(x2 + y2));
    if (x != 0 && y != 0 && z != 0) r -= x * y * z * atanq(y * z / (x * R));
    r += (2 * x2 - y2 - z2) * R / 6;
    return r;
}

static q_t newell_g(q_t x, q_t y, q_t z)
{
    q_t sgn = 1;                                              /* g is odd in x and y, even in z */
    if (x < 0) { x = -x; sgn = -sgn; }
    if (y < 0) { y = -y; sgn = -sgn; }
    z = fabsq(z);
    q_t x2 = x * x, y2 = y * y, z2 = z * z, R = sqrtq(x2 + y2 + z2), r = 0;
    if (x == 0 || y == 0) return 0;
    if (z != 0) r += x * y * z * asinhq(z / sqrtq(x2 + y2));
    if (y2 + z2 != 0) r += (y / 6) * (3 * z2 - y2) * asinhq(x / sqrtq(y2 + z2));
    if (x2 + z2 != 0) r += (x / 6) * (3 * z2 - x2) * asinhq(y / sqrtq(x2 + z2));
    if (z != 0) {
        r -= (z * z2 / 6) * atanq(x * y / (z * R));
        r -= (z * y2 / 2) * atanq(x * z / (y * R));
        r -= (z * x2 / 2) * atanq(y * z / (x * R));
    }
    r -= x * y * R / 3;
    return sgn * r;
}

/* the six components expressed through f and g by permuting axes (comp: xx yy zz xy xz yz) */
static q_t primitive(int comp, q_t X, q_t Y, q_t Z)
{
    switch (comp) {
    case 0: return newell_f(X, Y, Z);
    case 1: return newell_f(Y, X, Z);
    case 2: return newell_f(Z, Y, X);
    case 3: return newell_g(X, Y, Z);
    case 4: return newell_g(X, Z, Y);
    default: return newell_g(Y, Z, X);
    }
}

/* Plain definition of one entry: the 27-term signed sum, every term evaluated on the spot. */
static q_t newell_entry_q(int comp, int i, int j, int k, const double* d)
{
    static const int w[3] = { 1, -2, 1 };
    q_t s = 0, dx = d[0], dy = d[1], dz = d[2];
    for (int a = -1; a <= 1; ++a)
        for (int b = -1; b <= 1; ++b)
            for (int c = -1; c <= 1; ++c)
                s += (q_t)(w[a + 1] * w[b + 1] * w[c + 1]) *
                     primitive(comp, (i + a) * dx, (j + b) * dy, (k + c) * dz);
    return -s / (4 * M_PIq * dx * dy * dz);
}

double orc_newell_entry(int comp, int i, int j, int k, const double* d)
{
    return (double)newell_entry_q(comp, i, j, k, d);
}

/* Lattice of primitives for one component over 0 <= i <= Lx etc. (index = |offset|; the sign of
 * odd components is restored on lookup), then the 27-point sums.  Same arithmetic as
 * newell_entry_q, the primitives just are not recomputed for neighbouring entries. */
typedef struct { int L[3]; q_t* v; int comp; } lattice;

static int comp_odd(int comp, int axis)
{
    static const int odd[6][3] = { {0,0,0}, {0,0,0}, {0,0,0}, {1,1,0}, {1,0,1}, {0,1,1} };
    return odd[comp][axis];
}

static q_t lat_get(const lattice* t, int i, int j, int k)
{
    q_t s = 1;
    if (i < 0) { i = -i; if (comp_odd(t->comp, 0)) s = -s; }
    if (j < 0) { j = -j; if (comp_odd(t->comp, 1)) s = -s; }
    if (k < 0) { k = -k; if (comp_odd(t->comp, 2)) s = -s; }
    return s * t->v[((int64_t)k * (t->L[1] + 1) + j) * (t->L[0] + 1) + i];
}

/* N_comp(i,j,k) for 0 <= i <= Dx, ... written to out[(k*(Dy+1)+j)*(Dx+1)+i] as __float128. */
static void newell_octant_q(int comp, const int* D, const double* d, q_t* out)
{
    lattice t;
    t.comp = comp;
    for (int a = 0; a < 3; ++a) t.L[a] = D[a] + 1;
    int64_t cnt = (int64_t)(t.L[0] + 1) * (t.L[1] + 1) * (t.L[2] + 1);
    t.v = (q_t*)malloc(sizeof(q_t) * cnt);
    q_t dx = d[0], dy = d[1], dz = d[2];
#pragma omp parallel for collapse(2) schedule(dynamic, 4)
    for (int k = 0; k <= t.L[2]; ++k)
        for (int j = 0; j <= t.L[1]; ++j)
            for (int i = 0; i <= t.L[0]; ++i)
                t.v[((int64_t)k * (t.L[1] + 1) + j) * (t.L[0] + 1) + i] =
                    primitive(comp, i * dx, j * dy, k * dz);
    static const int w[3] = { 1, -2, 1 };
#pragma omp parallel for collapse(2)
    for (int k = 0; k <= D[2]; ++k)
        for (int j = 0; j <= D[1]; ++j)
            for (int i = 0; i <= D[0]; ++i) {
                q_t s = 0;
                for (int a = -1; a <= 1; ++a)
                    for (int b = -1; b <= 1; ++b)
                        for (int c = -1; c <= 1; ++c)
                            s += (q_t)(w[a + 1] * w[b + 1] * w[c + 1]) * lat_get(&t, i + a, j + b, k + c);
                out[((int64_t)k * (D[1] + 1) + j) * (D[0] + 1) + i] = -s / (4 * M_PIq * dx * dy * dz);
            }
    free(t.v);
}

/* Interaction table K_comp(d) (readings A3, A4).
 *   open axis a    : signed offsets d_a in [-(n_a-1), n_a-1], table length T_a = 2 n_a - 1,
 *                    index d_a + n_a - 1.
 *   periodic axis a: circular index j_a = (r_a - r'_a) mod n_a, T_a = n_a; the offset is the minimum
 *                    image d_a in [-n_a/2, n_a/2] (the tie |d_a| = n_a/2 is the mean of both signs) and
 *                    K = sum_{q=-R_a..R_a} N(d + q n_a e_a).
 *   exactly two periodic axes + zero_mode != 0: each plane d_w of the open axis w gets the
 *                    constant that makes its plane sum equal t_ij(d_w) (t_ww(0) = 1, else 0).
 * out: [6][Tz][Ty][Tx] doubles.  Returns 0, or -1 on bad arguments.
 */
int orc_tensor_table(const int* n, const double* d, const int* periodic, const int* images,
                     int zero_mode, double* out)
{
    int T[3], D[3], R[3];
    for (int a = 0; a < 3; ++a) {
        if (n[a] < 1) return -1;
        R[a] = periodic[a] ? images[a] : 0;
        T[a] = periodic[a] ? n[a] : 2 * n[a] - 1;
        /* largest |offset| whose N is needed */
        D[a] = periodic[a] ? n[a] / 2 + R[a] * n[a] : n[a] - 1;
    }
    int64_t oct = (int64_t)(D[0] + 1) * (D[1] + 1) * (D[2] + 1);
    int64_t TT = (int64_t)T[0] * T[1] * T[2];
    q_t* N = (q_t*)malloc(sizeof(q_t) * oct);
    if (!N) return -1;
    for (int comp = 0; comp < 6; ++comp) {
        newell_octant_q(comp, D, d, N);
        lattice t = { { D[0], D[1], D[2] }, N, comp };      /* reuse the signed lookup */
#pragma omp parallel for collapse(2)
        for (int tz = 0; tz < T[2]; ++tz)
            for (int ty = 0; ty < T[1]; ++ty)
                for (int tx = 0; tx < T[0]; ++tx) {
                    int tt[3] = { tx, ty, tz }, lo[3], cnt[3];
                    /* candidate minimum-image offsets per axis: one, or two at the tie */
                    for (int a = 0; a < 3; ++a) {
                        if (!periodic[a]) { lo[a] = tt[a] - (n[a] - 1); cnt[a] = 1; }
                        else {
                            int j = tt[a];
                            if (2 * j < n[a]) { lo[a] = j; cnt[a] = 1; }
                            else if (2 * j > n[a]) { lo[a] = j - n[a]; cnt[a] = 1; }
                            else { lo[a] = -j; cnt[a] = 2; }      /* -n/2 and +n/2 */
                        }
                    }
                    q_t s = 0;
                    for (int ux = 0; ux < cnt[0]; ++ux)
                        for (int uy = 0; uy < cnt[1]; ++uy)
                            for (int uz = 0; uz < cnt[2]; ++uz) {
                                int d0[3] = { lo[0] + ux * n[0], lo[1] + uy * n[1], lo[2] + uz * n[2] };
                                q_t si = 0;
                                for (int qx = -R[0]; qx <= R[0]; ++qx)
                                    for (int qy = -R[1]; qy <= R[1]; ++qy)
                                        for (int qz = -R[2]; qz <= R[2]; ++qz)
                                            si += lat_get(&t, d0[0] + qx * n[0], d0[1] + qy * n[1],
                                                          d0[2] + qz * n[2]);
                                s += si / (cnt[0] * cnt[1] * cnt[2]);
                            }
                    out[(int64_t)comp * TT + ((int64_t)tz * T[1] + ty) * T[0] + tx] = (double)s;
                }
    }
    free(N);
    int np = periodic[0] + periodic[1] + periodic[2];
    if (zero_mode && np == 2) {
        int w = !periodic[0] ? 0 : (!periodic[1] ? 1 : 2);
        for (int comp = 0; comp < 6; ++comp) {
            int is_ww = (comp == w);                     /* comps 0,1,2 = xx,yy,zz */
            for (int tw = 0; tw < T[w]; ++tw) {
                int dw = tw - (n[w] - 1);
                long double plane = 0;
                int64_t cnt = 0;
                for (int tz = 0; tz < T[2]; ++tz)
                    for (int ty = 0; ty < T[1]; ++ty)
                        for (int tx = 0; tx < T[0]; ++tx) {
                            int tt[3] = { tx, ty, tz };
                            if (tt[w] != tw) continue;
                            plane += out[(int64_t)comp * TT + ((int64_t)tz * T[1] + ty) * T[0] + tx];
                            ++cnt;
                        }
                double target = (is_ww && dw == 0) ? 1.0 : 0.0;
                double c = (double)((target - plane) / cnt);
                for (int tz = 0; tz < T[2]; ++tz)
                    for (int ty = 0; ty < T[1]; ++ty)
                        for (int tx = 0; tx < T[0]; ++tx) {
                            int tt[3] = { tx, ty, tz };
                            if (tt[w] != tw) continue;
                            out[(int64_t)comp * TT + ((int64_t)tz * T[1] + ty) * T[0] + tx] += c;
                        }
            }
        }
    }
    if (zero_mode && np == 3) {
        /* fully periodic box (reading A4, last case): the k = 0 mode of every component is set to 0 by removing the
         * mean of the image-summed table, i.e. a uniformly polarised periodic crystal feels no field
         * (short-circuit electrical boundary conditions). */
        for (int comp = 0; comp < 6; ++comp) {
            long double sum = 0;
            for (int64_t i = 0; i < TT; ++i) sum += out[(int64_t)comp * TT + i];
            double mean = (double)(sum / TT);
            for (int64_t i = 0; i < TT; ++i) out[(int64_t)comp * TT + i] -= mean;
        }
    }
    return 0;
}

/* index of the table entry for the ordered pair (target r, source r') along one axis */
static inline int pair_index(int r, int rp, int n, int periodic)
{
    return periodic ? (((r - rp) % n) + n) % n : r - rp + n - 1;
}

/* E_i(r) = -scale * sum_{r'} sum_j K_ij(r - r') P_j(r'), scale = 1/(eps0 epsB); every cell pair,
 * r' = r included (Eq. 5-6 applied to cell-wise constant P).  Targets: all cells, or the listed
 * ones (ntargets > 0: targets[] holds linear cell indices, E is [3][ntargets]). */
void orc_field_direct(const int* n, const int* periodic, const double* K, const double* P,
                      double scale, int64_t ntargets, const int64_t* targets, double* E)
{
    static const int cidx[3][3] = { { 0, 3, 4 }, { 3, 1, 5 }, { 4, 5, 2 } };
    int T[3];
    for (int a = 0; a < 3; ++a) T[a] = periodic[a] ? n[a] : 2 * n[a] - 1;
    int64_t TT = (int64_t)T[0] * T[1] * T[2];
    int64_t N = (int64_t)n[0] * n[1] * n[2];
    int64_t M = ntargets > 0 ? ntargets : N;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t t = 0; t < M; ++t) {
        int64_t r = ntargets > 0 ? targets[t] : t;
        int x = (int)(r % n[0]), y = (int)((r / n[0]) % n[1]), z = (int)(r / ((int64_t)n[0] * n[1]));
        long double acc[3] = { 0, 0, 0 };
        for (int zp = 0; zp < n[2]; ++zp)
            for (int yp = 0; yp < n[1]; ++yp)
                for (int xp = 0; xp < n[0]; ++xp) {
                    int64_t rp = ((int64_t)zp * n[1] + yp) * n[0] + xp;
                    int64_t e = ((int64_t)pair_index(z, zp, n[2], periodic[2]) * T[1] +
                                 pair_index(y, yp, n[1], periodic[1])) * T[0] +
                                pair_index(x, xp, n[0], periodic[0]);
                    for (int i = 0; i < 3; ++i)
                        for (int j = 0; j < 3; ++j)
                            acc[i] += (long double)K[cidx[i][j] * TT + e] * P[(int64_t)j * N + rp];
                }
        for (int i = 0; i < 3; ++i) E[(int64_t)i * M + t] = (double)(-scale * acc[i]);
    }
}
