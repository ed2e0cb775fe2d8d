/*
 * demag_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU oracle for the demagnetizing-field convolution of
 * arXiv 2308.08447 (Section II, Eq. (1)):
 *
 *        H_d,i = - sum_j N(i-j) M_j          (sum over all mesh points, j = i included)
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load this library.  It shares no code with paper_2308_08447_b200/csrc (the CUDA path).
 *
 * What is here (each function cites the passage it follows):
 *   newell_f / newell_g / oracle_newell_N   closed-form cell-averaged tensor ("formulas in
 *                                           Ref. [23]"; reading R1)
 *   oracle_quad_N                           Gauss-Legendre quadrature of the tent-weighted
 *                                           dipole kernel = the integral DEFINITION of N
 *                                           (reading R4, far field)
 *   oracle_tensor_table                     N over non-negative offsets, near = Newell,
 *                                           far = quadrature
 *   oracle_direct_sum (O-A)                 Eq. (1) written out, Kahan-compensated
 *   oracle_direct_sum_sampled (O-S)         Eq. (1) at selected cells only
 *   oracle_naive_dft_conv (O-B)             zero-padded convolution through O(N^2) DFTs
 *                                           (PAPER.md:27 "convolution theorem", :31-35 padding)
 *
 * Parity pins live in tests/test_oracle_pins.py; none of these functions is "parity unpinned".
 *
 * Array conventions (reading R8): planar [component][z][y][x], x fastest.
 * Tensor component order: xx, yy, zz, xy, xz, yz.
 * OpenMP is used only to split independent OUTPUT cells across threads; the arithmetic of
 * each output is the plain definition.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <complex.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PI 3.14159265358979323846264338327950288

/* ------------------------------------------------------------------------------------------
 * Newell closed form (Newell, Williams, Dunlop 1993 = Ref. [23] of the paper).
 * f is even in x,y,z.  g is odd in x and y, even in z.  Terms whose prefactor vanishes are
 * dropped (their transcendental argument is 0/0 there).
 * ---------------------------------------------------------------------------------------- */
static double newell_f(double x, double y, double z)
{
    x = fabs(x); y = fabs(y); z = fabs(z);
    const double x2 = x * x, y2 = y * y, z2 = z * z;
    const double R = sqrt(x2 + y2 + z2);
    if (R == 0.0) return 0.0;
    double s = 0.0, c;
    c = 0.5 * y * (z2 - x2); if (c != 0.0) s += c * asinh(y / sqrt(x2 + z2));
    c = 0.5 * z * (y2 - x2); if (c != 0.0) s += c * asinh(z / sqrt(x2 + y2));
    c = x * y * z;           if (c != 0.0) s -= c * atan(y * z / (x * R));
    s += (2.0 * x2 - y2 - z2) * R / 6.0;
    return s;
}

static double newell_g(double x, double y, double z)
{
    if (x == 0.0 || y == 0.0) return 0.0;
    const double sgn = ((x < 0.0) != (y < 0.0)) ? -1.0 : 1.0;
    x = fabs(x); y = fabs(y); z = fabs(z);
    const double x2 = x * x, y2 = y * y, z2 = z * z;
    const double R = sqrt(x2 + y2 + z2);
    double s = 0.0, c;
    c = x * y * z;                     if (c != 0.0) s += c * asinh(z / sqrt(x2 + y2));
    c = (y / 6.0) * (3.0 * z2 - y2);   if (c != 0.0) s += c * asinh(x / sqrt(y2 + z2));
    c = (x / 6.0) * (3.0 * z2 - x2);   if (c != 0.0) s += c * asinh(y / sqrt(x2 + z2));
    c = z * z2 / 6.0;                  if (c != 0.0) s -= c * atan(x * y / (z * R));
    c = z * y2 / 2.0;                  if (c != 0.0) s -= c * atan(x * z / (y * R));
    c = z * x2 / 2.0;                  if (c != 0.0) s -= c * atan(y * z / (x * R));
    s -= x * y * R / 3.0;
    return sgn * s;
}

/* 27-point tensor-product second difference  d2_x d2_y d2_z phi  (weights 1,-2,1 per axis). */
static double stencil27(double (*phi)(double, double, double),
                        double X, double Y, double Z, double hx, double hy, double hz)
{
    static const double w[3] = {1.0, -2.0, 1.0};
    double s = 0.0;
    for (int a = -1; a <= 1; ++a)
        for (int b = -1; b <= 1; ++b)
            for (int c = -1; c <= 1; ++c)
                s += w[a + 1] * w[b + 1] * w[c + 1] * phi(X + a * hx, Y + b * hy, Z + c * hz);
    return s;
}

static double newell_Nxx(double X, double Y, double Z, double hx, double hy, double hz)
{
    return -stencil27(newell_f, X, Y, Z, hx, hy, hz) / (4.0 * PI * hx * hy * hz);
}
static double newell_Nxy(double X, double Y, double Z, double hx, double hy, double hz)
{
    return -stencil27(newell_g, X, Y, Z, hx, hy, hz) / (4.0 * PI * hx * hy * hz);
}

/* All six components at offset (X,Y,Z) [metres] for cell (hx,hy,hz), closed form.
 * Nyy, Nzz, Nxz, Nyz follow from Nxx, Nxy by permuting the axes (R1). */
void oracle_newell_N(double X, double Y, double Z, double hx, double hy, double hz, double *N6)
{
    N6[0] = newell_Nxx(X, Y, Z, hx, hy, hz);
    N6[1] = newell_Nxx(Y, X, Z, hy, hx, hz);
    N6[2] = newell_Nxx(Z, Y, X, hz, hy, hx);
    N6[3] = newell_Nxy(X, Y, Z, hx, hy, hz);
    N6[4] = newell_Nxy(X, Z, Y, hx, hz, hy);
    N6[5] = newell_Nxy(Y, Z, X, hy, hz, hx);
}

/* ------------------------------------------------------------------------------------------
 * Integral definition of N for two identical, non-overlapping cuboids offset by r:
 *   N_ab(r) = V  INT  prod_c [ (1-|u_c|/h_c)/h_c ]  K_ab(r+u) d^3u ,  |u_c| <= h_c
 *   K_ab(p) = (1/4pi) ( delta_ab/p^3 - 3 p_a p_b / p^5 )
 * (the field of a dipole, averaged over source and target cell; R4).  Each axis is
 * split at u=0 and integrated with m-point Gauss-Legendre (m = 2,3,4,6,8).
 * ---------------------------------------------------------------------------------------- */
static int gauss_legendre_01(int m, double *t, double *w)
{
    /* nodes/weights on [-1,1], mapped to [0,1] below */
    double x[8], ww[8];
    switch (m) {
    case 2:
        x[0] = -sqrt(1.0 / 3.0); x[1] = -x[0]; ww[0] = ww[1] = 1.0; break;
    case 3:
        x[0] = -sqrt(0.6); x[1] = 0.0; x[2] = -x[0];
        ww[0] = ww[2] = 5.0 / 9.0; ww[1] = 8.0 / 9.0; break;
    case 4: {
        const double a = sqrt(3.0 / 7.0 - 2.0 / 7.0 * sqrt(1.2));
        const double b = sqrt(3.0 / 7.0 + 2.0 / 7.0 * sqrt(1.2));
        x[0] = -b; x[1] = -a; x[2] = a; x[3] = b;
        ww[0] = ww[3] = (18.0 - sqrt(30.0)) / 36.0;
        ww[1] = ww[2] = (18.0 + sqrt(30.0)) / 36.0; break; }
    default: {
        /* Newton iteration on the Legendre polynomial P_m (textbook construction). */
        if (m < 1 || m > 8) return -1;
        for (int i = 0; i < m; ++i) {
            double z = cos(PI * (i + 0.75) / (m + 0.5)), pp = 1.0;
            for (int it = 0; it < 100; ++it) {
                double p1 = 1.0, p2 = 0.0;
                for (int j = 1; j <= m; ++j) {
                    const double p3 = p2; p2 = p1;
                    p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j;
                }
                pp = m * (z * p1 - p2) / (z * z - 1.0);
                const double dz = p1 / pp; z -= dz;
                if (fabs(dz) < 1e-16) break;
            }
            x[i] = z; ww[i] = 2.0 / ((1.0 - z * z) * pp * pp);
        } }
    }
    for (int i = 0; i < m; ++i) { t[i] = 0.5 * (x[i] + 1.0); w[i] = 0.5 * ww[i]; }
    return 0;
}

void oracle_quad_N(double X, double Y, double Z, double hx, double hy, double hz, int m, double *N6)
{
    double t[8], w[8];
    double acc[6] = {0, 0, 0, 0, 0, 0};
    if (gauss_legendre_01(m, t, w) != 0) { for (int c = 0; c < 6; ++c) N6[c] = NAN; return; }
    /* signed nodes u = +-h t with weight w (1-t): the tent (1-|u|/h)/h du = (1-t) dt */
    for (int ix = 0; ix < 2 * m; ++ix) {
        const double tx = t[ix % m], wx = w[ix % m] * (1.0 - tx), ux = (ix < m ? tx : -tx) * hx;
        for (int iy = 0; iy < 2 * m; ++iy) {
            const double ty = t[iy % m], wy = w[iy % m] * (1.0 - ty), uy = (iy < m ? ty : -ty) * hy;
            for (int iz = 0; iz < 2 * m; ++iz) {
                const double tz = t[iz % m], wz = w[iz % m] * (1.0 - tz), uz = (iz < m ? tz : -tz) * hz;
                const double px = X + ux, py = Y + uy, pz = Z + uz;
                const double r2 = px * px + py * py + pz * pz;
                const double r = sqrt(r2), i3 = 1.0 / (r2 * r), i5 = 3.0 * i3 / r2;
                const double W = wx * wy * wz;
                acc[0] += W * (i3 - i5 * px * px);
                acc[1] += W * (i3 - i5 * py * py);
                acc[2] += W * (i3 - i5 * pz * pz);
                acc[3] += W * (-i5 * px * py);
                acc[4] += W * (-i5 * px * pz);
                acc[5] += W * (-i5 * py * pz);
            }
        }
    }
    const double V = hx * hy * hz;
    for (int c = 0; c < 6; ++c) N6[c] = acc[c] * V / (4.0 * PI);
}

/* Switch radii, in units of the largest cell edge (R4):
 *   |r| <= 16 max(h)          closed form (Newell)
 *   16 max(h) < |r| <= 128    quadrature, m = 3 nodes per half axis (error ~ (h/r)^6)
 *   |r| > 128 max(h)          quadrature, m = 2 (error ~ (h/r)^4 <= 4e-9 relative) */
#define ORACLE_R_NEWELL 16.0
#define ORACLE_R_M3 128.0

void oracle_N_at(double X, double Y, double Z, double hx, double hy, double hz, double *N6)
{
    const double hm = fmax(hx, fmax(hy, hz));
    const double r = sqrt(X * X + Y * Y + Z * Z) / hm;
    if (r <= ORACLE_R_NEWELL) oracle_newell_N(X, Y, Z, hx, hy, hz, N6);
    else if (r <= ORACLE_R_M3) oracle_quad_N(X, Y, Z, hx, hy, hz, 3, N6);
    else oracle_quad_N(X, Y, Z, hx, hy, hz, 2, N6);
}

/* Table over non-negative cell offsets d = (dx,dy,dz), 0 <= d_a < n_a:
 *   T[c][dz][dy][dx] = N_c(dx*hx, dy*hy, dz*hz).   (a0 of the scope table) */
void oracle_tensor_table(int nx, int ny, int nz, double hx, double hy, double hz, double *T)
{
    const size_t nc = (size_t)nx * ny * nz;
#pragma omp parallel for schedule(dynamic, 64) collapse(2)
    for (int dz = 0; dz < nz; ++dz)
        for (int dy = 0; dy < ny; ++dy)
            for (int dx = 0; dx < nx; ++dx) {
                double N6[6];
                oracle_N_at(dx * hx, dy * hy, dz * hz, hx, hy, hz, N6);
                const size_t o = ((size_t)dz * ny + dy) * nx + dx;
                for (int c = 0; c < 6; ++c) T[c * nc + o] = N6[c];
            }
}

/* ------------------------------------------------------------------------------------------
 * O-A: Eq. (1) written out.  N(-d) from the table by parity (diagonal even; xy odd in x,y;
 * xz odd in x,z; yz odd in y,z -- DESIGN.md R1).  Kahan-compensated accumulation.
 * ---------------------------------------------------------------------------------------- */
typedef struct { double s, c; } kahan_t;
static inline void kadd(kahan_t *k, double v)
{
    const double y = v - k->c, t = k->s + y;
    k->c = (t - k->s) - y; k->s = t;
}

static void direct_sum_cell(int nx, int ny, int nz, const double *T, const double *M,
                            int ix, int iy, int iz, double *H3)
{
    const size_t nc = (size_t)nx * ny * nz;
    kahan_t ax = {0, 0}, ay = {0, 0}, az = {0, 0};
    for (int jz = 0; jz < nz; ++jz) {
        const int dz = iz - jz, adz = abs(dz); const double sz = dz < 0 ? -1.0 : 1.0;
        for (int jy = 0; jy < ny; ++jy) {
            const int dy = iy - jy, ady = abs(dy); const double sy = dy < 0 ? -1.0 : 1.0;
            const size_t trow = ((size_t)adz * ny + ady) * nx;
            const size_t mrow = ((size_t)jz * ny + jy) * nx;
            for (int jx = 0; jx < nx; ++jx) {
                const int dx = ix - jx, adx = abs(dx); const double sx = dx < 0 ? -1.0 : 1.0;
                const size_t to = trow + adx, mo = mrow + jx;
                const double Nxx = T[to], Nyy = T[nc + to], Nzz = T[2 * nc + to];
                const double Nxy = sx * sy * T[3 * nc + to];
                const double Nxz = sx * sz * T[4 * nc + to];
                const double Nyz = sy * sz * T[5 * nc + to];
                const double mx = M[mo], my = M[nc + mo], mz = M[2 * nc + mo];
                kadd(&ax, Nxx * mx); kadd(&ax, Nxy * my); kadd(&ax, Nxz * mz);
                kadd(&ay, Nxy * mx); kadd(&ay, Nyy * my); kadd(&ay, Nyz * mz);
                kadd(&az, Nxz * mx); kadd(&az, Nyz * my); kadd(&az, Nzz * mz);
            }
        }
    }
    H3[0] = -ax.s; H3[1] = -ay.s; H3[2] = -az.s;
}

void oracle_direct_sum(int nx, int ny, int nz, const double *T, const double *M, double *H)
{
    const size_t nc = (size_t)nx * ny * nz;
#pragma omp parallel for schedule(dynamic, 16)
    for (long i = 0; i < (long)nc; ++i) {
        const int ix = (int)(i % nx), iy = (int)((i / nx) % ny), iz = (int)(i / ((size_t)nx * ny));
        double H3[3];
        direct_sum_cell(nx, ny, nz, T, M, ix, iy, iz, H3);
        H[i] = H3[0]; H[nc + i] = H3[1]; H[2 * nc + i] = H3[2];
    }
}

/* O-S: Eq. (1) at nsamp cells given as flat indices (iz*ny+iy)*nx+ix; Hs[s][3]. */
void oracle_direct_sum_sampled(int nx, int ny, int nz, const double *T, const double *M,
                               int nsamp, const long long *cells, double *Hs)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < nsamp; ++s) {
        const long long i = cells[s];
        const int ix = (int)(i % nx), iy = (int)((i / nx) % ny), iz = (int)(i / ((long long)nx * ny));
        direct_sum_cell(nx, ny, nz, T, M, ix, iy, iz, Hs + 3 * s);
    }
}

/* ------------------------------------------------------------------------------------------
 * O-B: zero-padded convolution through the convolution theorem, with every DFT
 * evaluated by its O(N^2) definition  X[k] = sum_j x[j] exp(-2 pi i (j k mod N)/N).
 * Padded sizes (Px,Py,Pz): P_a = 2 n_a for an open axis with n_a > 1, else n_a (
 * DESIGN.md R6).  Padded kernel: K[d] = N(s(d)) with s_a = d_a (d_a < n_a), d_a - P_a (d_a > n_a),
 * and 0 at d_a = n_a when P_a = 2 n_a.
 * ---------------------------------------------------------------------------------------- */
static void dft_axis(double complex *a, int Px, int Py, int Pz, int axis, int sign)
{
    const int P[3] = {Px, Py, Pz};
    const int N = P[axis];
    if (N == 1) return;
    const size_t stride = axis == 0 ? 1 : (axis == 1 ? (size_t)Px : (size_t)Px * Py);
    const size_t total = (size_t)Px * Py * Pz;
    const size_t nlines = total / N;
    double complex *tw = malloc(sizeof(double complex) * N);
    for (int k = 0; k < N; ++k) tw[k] = cexp(sign * 2.0 * PI * I * (double)k / (double)N);
#pragma omp parallel
    {
        double complex *buf = malloc(sizeof(double complex) * N);
#pragma omp for schedule(static)
        for (long l = 0; l < (long)nlines; ++l) {
            /* base offset of line l: enumerate the two other axes */
            size_t base;
            if (axis == 0) base = (size_t)l * Px;
            else if (axis == 1) base = ((size_t)l / Px) * ((size_t)Px * Py) + ((size_t)l % Px);
            else base = (size_t)l;
            for (int k = 0; k < N; ++k) {
                double complex s = 0.0;
                for (int j = 0; j < N; ++j) s += a[base + j * stride] * tw[(int)(((long)j * k) % N)];
                buf[k] = s;
            }
            for (int k = 0; k < N; ++k) a[base + k * stride] = buf[k];
        }
        free(buf);
    }
    free(tw);
}

static void dft3(double complex *a, int Px, int Py, int Pz, int sign)
{
    dft_axis(a, Px, Py, Pz, 0, sign);
    dft_axis(a, Px, Py, Pz, 1, sign);
    dft_axis(a, Px, Py, Pz, 2, sign);
}

int oracle_naive_dft_conv(int nx, int ny, int nz, int Px, int Py, int Pz,
                          const double *T, const double *M, double *H)
{
    const int n[3] = {nx, ny, nz}, P[3] = {Px, Py, Pz};
    for (int a = 0; a < 3; ++a) if (!(P[a] == n[a] || P[a] >= 2 * n[a] - 1)) return -1;
    const size_t nc = (size_t)nx * ny * nz, np = (size_t)Px * Py * Pz;
    double complex *K = calloc(6 * np, sizeof(double complex));
    double complex *Mp = calloc(3 * np, sizeof(double complex));
    double complex *Hp = calloc(3 * np, sizeof(double complex));
    if (!K || !Mp || !Hp) { free(K); free(Mp); free(Hp); return -2; }
    /* parity of component c along axis a: -1 if odd */
    static const int par[6][3] = {{1, 1, 1}, {1, 1, 1}, {1, 1, 1}, {-1, -1, 1}, {-1, 1, -1}, {1, -1, -1}};
    for (int dz = 0; dz < Pz; ++dz)
        for (int dy = 0; dy < Py; ++dy)
            for (int dx = 0; dx < Px; ++dx) {
                const int d[3] = {dx, dy, dz};
                int s[3], ok = 1;
                for (int a = 0; a < 3; ++a) {
                    if (d[a] < n[a]) s[a] = d[a];
                    else if (P[a] - d[a] < n[a] && P[a] - d[a] > 0) s[a] = d[a] - P[a];
                    else ok = 0;                          /* the never-addressed slot(s): 0 */
                }
                if (!ok) continue;
                const size_t to = ((size_t)abs(s[2]) * ny + abs(s[1])) * nx + abs(s[0]);
                const size_t po = ((size_t)dz * Py + dy) * Px + dx;
                for (int c = 0; c < 6; ++c) {
                    double sg = 1.0;
                    for (int a = 0; a < 3; ++a) if (s[a] < 0 && par[c][a] < 0) sg = -sg;
                    K[c * np + po] = sg * T[c * nc + to];
                }
            }
    for (int c = 0; c < 3; ++c)
        for (int z = 0; z < nz; ++z)
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x)
                    Mp[c * np + ((size_t)z * Py + y) * Px + x] = M[c * nc + ((size_t)z * ny + y) * nx + x];
    for (int c = 0; c < 6; ++c) dft3(K + c * np, Px, Py, Pz, -1);
    for (int c = 0; c < 3; ++c) dft3(Mp + c * np, Px, Py, Pz, -1);
    for (size_t p = 0; p < np; ++p) {
        const double complex mx = Mp[p], my = Mp[np + p], mz = Mp[2 * np + p];
        const double complex kxx = K[p], kyy = K[np + p], kzz = K[2 * np + p];
        const double complex kxy = K[3 * np + p], kxz = K[4 * np + p], kyz = K[5 * np + p];
        Hp[p]          = -(kxx * mx + kxy * my + kxz * mz);
        Hp[np + p]     = -(kxy * mx + kyy * my + kyz * mz);
        Hp[2 * np + p] = -(kxz * mx + kyz * my + kzz * mz);
    }
    for (int c = 0; c < 3; ++c) dft3(Hp + c * np, Px, Py, Pz, +1);
    const double scale = 1.0 / (double)np;
    for (int c = 0; c < 3; ++c)
        for (int z = 0; z < nz; ++z)
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x)
                    H[c * nc + ((size_t)z * ny + y) * nx + x] =
                        creal(Hp[c * np + ((size_t)z * Py + y) * Px + x]) * scale;
    free(K); free(Mp); free(Hp);
    return 0;
}

/* The transformed kernel itself (for checking that it is real, "packed using y
 * and z axis symmetries"): returns max |Im K^| / max |Re K^| over all six components. */
double oracle_kernel_spectrum_imag_ratio(int nx, int ny, int nz, int Px, int Py, int Pz, const double *T)
{
    const int n[3] = {nx, ny, nz}, P[3] = {Px, Py, Pz};
    const size_t nc = (size_t)nx * ny * nz, np = (size_t)Px * Py * Pz;
    static const int par[6][3] = {{1, 1, 1}, {1, 1, 1}, {1, 1, 1}, {-1, -1, 1}, {-1, 1, -1}, {1, -1, -1}};
    double complex *K = calloc(6 * np, sizeof(double complex));
    for (int dz = 0; dz < Pz; ++dz)
        for (int dy = 0; dy < Py; ++dy)
            for (int dx = 0; dx < Px; ++dx) {
                const int d[3] = {dx, dy, dz};
                int s[3], ok = 1;
                for (int a = 0; a < 3; ++a) {
                    if (d[a] < n[a]) s[a] = d[a];
                    else if (P[a] - d[a] < n[a] && P[a] - d[a] > 0) s[a] = d[a] - P[a];
                    else ok = 0;
                }
                if (!ok) continue;
                const size_t to = ((size_t)abs(s[2]) * ny + abs(s[1])) * nx + abs(s[0]);
                const size_t po = ((size_t)dz * Py + dy) * Px + dx;
                for (int c = 0; c < 6; ++c) {
                    double sg = 1.0;
                    for (int a = 0; a < 3; ++a) if (s[a] < 0 && par[c][a] < 0) sg = -sg;
                    K[c * np + po] = sg * T[c * nc + to];
                }
            }
    double mre = 0.0, mim = 0.0;
    for (int c = 0; c < 6; ++c) {
        dft3(K + c * np, Px, Py, Pz, -1);
        for (size_t p = 0; p < np; ++p) {
            mre = fmax(mre, fabs(creal(K[c * np + p])));
            mim = fmax(mim, fabs(cimag(K[c * np + p])));
        }
    }
    free(K);
    return mim / mre;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
