// builder.cuh -- plan-time code (scope row a0): the demagnetizing tensor N in fp64 and its
// real-valued half spectrum (PAPER.md:27 "N ... computed using the formulas in Ref. [23]"; :35 "The
// kernel is computed in the initialization stage"; :255-256 packed by the y and z symmetries).
//
//   k_tensor_table  N_c(dx*hx, dy*hy, dz*hz) for 0 <= d_a < n_a:  closed form (Newell) within 24 cell
//                   edges, beyond that the Cartesian multipole series of the cell-averaged dipole
//                   kernel through h^4 (R4 -- deliberately NOT the oracle's quadrature).
//   k_sym_axis      one axis of the 3D transform of the even/odd extended tensor: the extension is
//                   synthesised on load, a complex fp64 FFT runs in shared memory, and only the real
//                   (even axis) or imaginary (odd axis) part of bins 0..N/2 is kept -- every partial
//                   result stays real, which is why the spectrum can be stored as real arrays.
//   k_pack_kernel   fold -1/(Nx Ny Nz) and the (i)^2 = -1 of two odd axes, transpose to
//                   [kx][kz'][ky'] and round once to the plan's precision (R3, R7).
#pragma once
#include "fft_core.cuh"

namespace demag {

// ---------------------------------------------------------------- closed form (near field), fp64
__device__ inline double nw_f(double x, double y, double z)
{
    x = fabs(x); y = fabs(y); z = fabs(z);
    const double x2 = x * x, y2 = y * y, z2 = z * z, R = sqrt(x2 + y2 + z2);
    if (R == 0.0) return 0.0;
    double s = (2.0 * x2 - y2 - z2) * R * (1.0 / 6.0);
    double c = 0.5 * y * (z2 - x2); if (c != 0.0) s += c * asinh(y / sqrt(x2 + z2));
    c = 0.5 * z * (y2 - x2);        if (c != 0.0) s += c * asinh(z / sqrt(x2 + y2));
    c = x * y * z;                  if (c != 0.0) s -= c * atan(y * z / (x * R));
    return s;
}
__device__ inline double nw_g(double x, double y, double z)
{
    if (x == 0.0 || y == 0.0) return 0.0;
    const double sg = ((x < 0.0) != (y < 0.0)) ? -1.0 : 1.0;
    x = fabs(x); y = fabs(y); z = fabs(z);
    const double x2 = x * x, y2 = y * y, z2 = z * z, R = sqrt(x2 + y2 + z2);
    double s = -x * y * R * (1.0 / 3.0);
    double c = x * y * z;                  if (c != 0.0) s += c * asinh(z / sqrt(x2 + y2));
    c = y * (3.0 * z2 - y2) * (1.0 / 6.0); if (c != 0.0) s += c * asinh(x / sqrt(y2 + z2));
    c = x * (3.0 * z2 - x2) * (1.0 / 6.0); if (c != 0.0) s += c * asinh(y / sqrt(x2 + z2));
    c = z * z2 * (1.0 / 6.0);              if (c != 0.0) s -= c * atan(x * y / (z * R));
    c = 0.5 * z * y2;                      if (c != 0.0) s -= c * atan(x * z / (y * R));
    c = 0.5 * z * x2;                      if (c != 0.0) s -= c * atan(y * z / (x * R));
    return sg * s;
}
template <bool G>
__device__ inline double nw_stencil(double X, double Y, double Z, double hx, double hy, double hz)
{
    double s = 0.0;
#pragma unroll 1
    for (int a = -1; a <= 1; ++a)
#pragma unroll 1
        for (int b = -1; b <= 1; ++b)
#pragma unroll 1
            for (int c = -1; c <= 1; ++c) {
                const double w = (a == 0 ? -2.0 : 1.0) * (b == 0 ? -2.0 : 1.0) * (c == 0 ? -2.0 : 1.0);
                s += w * (G ? nw_g(X + a * hx, Y + b * hy, Z + c * hz) : nw_f(X + a * hx, Y + b * hy, Z + c * hz));
            }
    return -s / (4.0 * 3.14159265358979323846 * hx * hy * hz);
}

// ---------------------------------------------------------------- multipole series (far field), fp64
// D[i][j][k] = d^i_x d^j_y d^k_z (1/rho), i+j+k <= 6, by the McMurchie-Davidson-type recursion
//   R^(m)_000 = (-1)^m (2m-1)!! / rho^(2m+1),   R^(m)_{i+1,j,k} = i R^(m+1)_{i-1,j,k} + x R^(m+1)_{i,j,k}.
struct Deriv6 {
    double v[7][7][7];
};
__device__ inline void deriv_inv_r(double x, double y, double z, Deriv6& D)
{
    // work array Rm[m][i][j][k] collapsed: we build for m = 6 down to 0, keeping only orders <= 6 - m
    double g[7];
    const double r2 = x * x + y * y + z * z, ir = rsqrt(r2), ir2 = 1.0 / r2;
    g[0] = ir;
    for (int m = 1; m <= 6; ++m) g[m] = -g[m - 1] * (2 * m - 1) * ir2;
    double cur[7][7][7], nxt[7][7][7];
    for (int m = 6; m >= 0; --m) {
        const int ord = 6 - m;
        // nxt holds R^(m+1) up to order ord-1
        for (int i = 0; i <= ord; ++i)
            for (int j = 0; i + j <= ord; ++j)
                for (int k = 0; i + j + k <= ord; ++k) {
                    double val;
                    if (i + j + k == 0) val = g[m];
                    else if (i > 0) val = (i > 1 ? (i - 1) * nxt[i - 2][j][k] : 0.0) + x * nxt[i - 1][j][k];
                    else if (j > 0) val = (j > 1 ? (j - 1) * nxt[i][j - 2][k] : 0.0) + y * nxt[i][j - 1][k];
                    else            val = (k > 1 ? (k - 1) * nxt[i][j][k - 2] : 0.0) + z * nxt[i][j][k - 1];
                    cur[i][j][k] = val;
                }
        for (int i = 0; i <= ord; ++i)
            for (int j = 0; i + j <= ord; ++j)
                for (int k = 0; i + j + k <= ord; ++k) nxt[i][j][k] = cur[i][j][k];
    }
    for (int i = 0; i <= 6; ++i)
        for (int j = 0; i + j <= 6; ++j)
            for (int k = 0; i + j + k <= 6; ++k) D.v[i][j][k] = nxt[i][j][k];
}

// N_ab = -(V/4pi) [ D_ab + (1/12) sum_c h_c^2 D_ab,cc + (1/360) sum_c h_c^4 D_ab,cccc
//                   + (1/144) sum_{c<d} h_c^2 h_d^2 D_ab,ccdd ]        (tent moments h^2/6, h^4/15)
__device__ inline void series_N(double X, double Y, double Z, double hx, double hy, double hz, double* N6)
{
    Deriv6 D;
    deriv_inv_r(X, Y, Z, D);
    const double h2[3] = {hx * hx, hy * hy, hz * hz};
    const int ab[6][3] = {{2, 0, 0}, {0, 2, 0}, {0, 0, 2}, {1, 1, 0}, {1, 0, 1}, {0, 1, 1}};
    const double pref = -hx * hy * hz / (4.0 * 3.14159265358979323846);
    for (int c6 = 0; c6 < 6; ++c6) {
        const int i = ab[c6][0], j = ab[c6][1], k = ab[c6][2];
        double s = D.v[i][j][k];
        s += (1.0 / 12.0) * (h2[0] * D.v[i + 2][j][k] + h2[1] * D.v[i][j + 2][k] + h2[2] * D.v[i][j][k + 2]);
        s += (1.0 / 360.0) * (h2[0] * h2[0] * D.v[i + 4][j][k] + h2[1] * h2[1] * D.v[i][j + 4][k] + h2[2] * h2[2] * D.v[i][j][k + 4]);
        s += (1.0 / 144.0) * (h2[0] * h2[1] * D.v[i + 2][j + 2][k] + h2[0] * h2[2] * D.v[i + 2][j][k + 2] + h2[1] * h2[2] * D.v[i][j + 2][k + 2]);
        N6[c6] = pref * s;
    }
}

#define DEMAG_BUILDER_R_NEAR 24.0

__device__ inline void tensor_at(double X, double Y, double Z, double hx, double hy, double hz, double* N6)
{
    const double hm = fmax(hx, fmax(hy, hz));
    if (sqrt(X * X + Y * Y + Z * Z) <= DEMAG_BUILDER_R_NEAR * hm) {
        N6[0] = nw_stencil<false>(X, Y, Z, hx, hy, hz);
        N6[1] = nw_stencil<false>(Y, X, Z, hy, hx, hz);
        N6[2] = nw_stencil<false>(Z, Y, X, hz, hy, hx);
        N6[3] = nw_stencil<true>(X, Y, Z, hx, hy, hz);
        N6[4] = nw_stencil<true>(X, Z, Y, hx, hz, hy);
        N6[5] = nw_stencil<true>(Y, Z, X, hy, hz, hx);
    } else {
        series_N(X, Y, Z, hx, hy, hz, N6);
    }
}

__global__ void __launch_bounds__(128) k_tensor_table(int nx, int ny, int nz, double hx, double hy, double hz,
                                                      double* __restrict__ T)
{
    const size_t nc = (size_t)nx * ny * nz;
    const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    if (i >= nc) return;
    const int dx = (int)(i % nx), dy = (int)((i / nx) % ny), dz = (int)(i / ((size_t)nx * ny));
    double N6[6];
    tensor_at(dx * hx, dy * hy, dz * hz, hx, hy, hz, N6);
    for (int c = 0; c < 6; ++c) T[c * nc + i] = N6[c];
}

// Periodic axes ("modified convolution kernel"; R11): the open-boundary tensor summed over
// `img` periodic images on each side of every periodic axis a (period n_a h_a), and the result symmetrised,
//   T(d) = sym_a [ sum_{|m_a| <= img} N((d_a + m_a n_a) h_a) ],   sym_a f(d_a) = ( f(d_a) + parity_a f(n_a - d_a) ) / 2,
// (indices mod n_a, so d_a = 0 maps to itself) because a periodic kernel obeys K(n_a - d_a) = parity_a K(d_a) and the
// truncated sum does so only up to its last images.  Since parity_a N(-x) = N(x), for d_a > 0 the symmetrised sum is the
// image sum over m_a = -img-1 .. img with weight 1/2 on the two end images; for d_a = 0 it is the plain sum over
// |m_a| <= img.  That is what the loops below evaluate.  img[a] < 0 marks an open axis (m_a = 0 only).
__global__ void __launch_bounds__(128) k_tensor_table_pbc(int nx, int ny, int nz, double hx, double hy, double hz,
                                                          int ix, int iy, int iz, double* __restrict__ T)
{
    const size_t nc = (size_t)nx * ny * nz;
    const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    if (i >= nc) return;
    const int dx = (int)(i % nx), dy = (int)((i / nx) % ny), dz = (int)(i / ((size_t)nx * ny));
    const bool ex = ix >= 0 && dx > 0, ey = iy >= 0 && dy > 0, ez = iz >= 0 && dz > 0;   // half-weight end images
    const int x0 = ix < 0 ? 0 : -ix - (ex ? 1 : 0), x1 = ix < 0 ? 0 : ix;
    const int y0 = iy < 0 ? 0 : -iy - (ey ? 1 : 0), y1 = iy < 0 ? 0 : iy;
    const int z0 = iz < 0 ? 0 : -iz - (ez ? 1 : 0), z1 = iz < 0 ? 0 : iz;
    double acc[6] = {0, 0, 0, 0, 0, 0};
    for (int mz = z0; mz <= z1; ++mz) {
        const double wz = (ez && (mz == z0 || mz == z1)) ? 0.5 : 1.0;
        for (int my = y0; my <= y1; ++my) {
            const double wy = wz * ((ey && (my == y0 || my == y1)) ? 0.5 : 1.0);
            for (int mx = x0; mx <= x1; ++mx) {
                const double w = wy * ((ex && (mx == x0 || mx == x1)) ? 0.5 : 1.0);
                double N6[6];
                tensor_at((dx + (double)mx * nx) * hx, (dy + (double)my * ny) * hy, (dz + (double)mz * nz) * hz, hx, hy, hz, N6);
                for (int c = 0; c < 6; ++c) acc[c] += w * N6[c];
            }
        }
    }
    for (int c = 0; c < 6; ++c) T[c * nc + i] = acc[c];
}

// ---------------------------------------------------------------- spectrum of the extended tensor
// Lines along one axis of a real fp64 array.  Line (o, i): element e at  o*so + i + e*se  (input and
// output use their own so/se).  The input line has n entries (offsets 0..n-1); it is extended to
// length N = 2^lN:  ext[e] = in[e] (e<n), 0 (e==n), par*in[N-e] (e>n)   (N == n: no extension).
// Output bins k = 0..nout-1 (nout = N/2+1): Re X[k] if par > 0, Im X[k] if par < 0.
// Tile = B adjacent inner indices i; smem s[N][B].
__global__ void __launch_bounds__(512) k_sym_axis(const double* __restrict__ in, double* __restrict__ out,
                                                  int n, int lN, int nout, int par, int ni, int B,
                                                  size_t so_in, size_t se_in, size_t so_out, size_t se_out,
                                                  const double2* __restrict__ tw)
{
    double2* s = reinterpret_cast<double2*>(demag_smem);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int N = 1 << lN;
    const int tilesI = (ni + B - 1) / B;
    const int it = blockIdx.x % tilesI;
    const size_t o = blockIdx.x / tilesI;
    const int i0 = it * B;
    const double* src = in + o * so_in + i0;
    for (int idx = tid; idx < N * B; idx += nthr) {
        const int b = idx % B, e = idx / B;
        double v = 0.0;
        if (i0 + b < ni) {
            if (e < n) v = src[(size_t)e * se_in + b];
            else if (N != n && e > n) v = par * src[(size_t)(N - e) * se_in + b];
        }
        s[swz<3>(e * B + b)] = make_double2(v, 0.0);
    }
    __syncthreads();
    fft_tile<double, false, true>(s, lN, B, B, tw, 0, tid, nthr);
    double* dst = out + o * so_out + i0;
    for (int idx = tid; idx < nout * B; idx += nthr) {
        const int b = idx % B, k = idx / B;
        if (i0 + b < ni) {
            const double2 v = s[swz<3>(pos_of_freq(k, lN) * B + b)];
            dst[(size_t)k * se_out + b] = par > 0 ? v.x : v.y;
        }
    }
}

// The same for a line too long for a complex tile (N = 16384: the x axis of nx = 8192 meshes): the real extended
// sequence is packed into N/2 complex points z[m] = ext[2m] + i ext[2m+1], transformed with a length-N/2 FFT and split,
//     X[k] = E[k] + w_N^k O[k],  E = (Z[k] + conj Z[N/2-k]) / 2,  O = -i (Z[k] - conj Z[N/2-k]) / 2.
// One line per block (B = 1), N > n (an extended axis); tw = exp(-2 pi i k / N).
__global__ void __launch_bounds__(512) k_sym_axis_packed(const double* __restrict__ in, double* __restrict__ out,
                                                         int n, int lN, int nout, int par, int ni,
                                                         size_t so_in, size_t se_in, size_t so_out, size_t se_out,
                                                         const double2* __restrict__ tw)
{
    double2* s = reinterpret_cast<double2*>(demag_smem);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int N = 1 << lN, Nh = N >> 1;
    const int i = blockIdx.x % ni;
    const size_t o = blockIdx.x / ni;
    const double* src = in + o * so_in + i;
    auto ext = [&](int e) -> double {
        if (e < n) return src[(size_t)e * se_in];
        if (e == n) return 0.0;
        return par * src[(size_t)(N - e) * se_in];
    };
    for (int m = tid; m < Nh; m += nthr) s[swz<3>(m)] = make_double2(ext(2 * m), ext(2 * m + 1));
    __syncthreads();
    fft_tile<double, false, true>(s, lN - 1, 1, 1, tw, 1, tid, nthr);
    double* dst = out + o * so_out + i;
    for (int k = tid; k < nout; k += nthr) {
        const double2 a = s[swz<3>(pos_of_freq(k & (Nh - 1), lN - 1))];
        double2 b = s[swz<3>(pos_of_freq((Nh - k) & (Nh - 1), lN - 1))];
        b.y = -b.y;                                                    // conj Z[N/2 - k]
        const double er = 0.5 * (a.x + b.x), ei = 0.5 * (a.y + b.y);
        const double dr = 0.5 * (a.x - b.x), di = 0.5 * (a.y - b.y);   // (Z - conj Z') / 2;  O = -i d = (di, -dr)
        const double orr = di, oi = -dr;
        const double2 w = k == Nh ? make_double2(-1.0, 0.0) : tw[k];
        const double xr = er + w.x * orr - w.y * oi, xi = ei + w.x * oi + w.y * orr;
        dst[(size_t)k * se_out] = par > 0 ? xr : xi;
    }
}

// K[kx][kz'][py] = sign_y * scale * A[kz'][ky'][kx],  ky = freq_of_pos(py), ky' = min(ky, Ny-ky),
// sign_y = -1 on mirrored ky of a component that is odd in y (the y axis is stored unpacked, in the
// digit-reversed "position" order in which the y FFT leaves W2, so the hot path never permutes).
template <typename T>
__global__ void k_pack_kernel(const double* __restrict__ A, T* __restrict__ K, int hx, int kpy, int kpz,
                              int Ny, int lNy, int par_y, double scale)
{
    const size_t n = (size_t)hx * kpz * Ny;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int py = (int)(i % Ny), kz = (int)((i / Ny) % kpz), kx = (int)(i / ((size_t)Ny * kpz));
        const int ky = freq_of_pos(py, lNy);
        const bool my = 2 * ky > Ny;
        const int kyp = my ? Ny - ky : ky;
        const double sg = (my && par_y < 0) ? -1.0 : 1.0;
        K[i] = (T)(sg * scale * A[((size_t)kz * kpy + kyp) * hx + kx]);
    }
}

}  // namespace demag
