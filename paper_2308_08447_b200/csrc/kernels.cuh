// kernels.cuh -- the hot-path kernels of demag_apply (scope rows a1..a8 of SURVEY.md section 8):
//   k_x_r2c   x real-to-complex FFT fused with zero padding and the xy transposition
//             (PAPER.md:35, :296-300 xFFT_R2C; :343 "xy transposition ... to avoid strided y FFTs")
//   k_y_fwd   y FFT, zero padding synthesised on load            (PAPER.md:309-315 yFFT)
//   k_z_mul   z FFT . kernel multiplication . z IFFT in one routine
//   k_y_inv   y IFFT fused with the crop
//   k_x_c2r   x complex-to-real IFFT fused with the crop, writes H
//   k_energy, k_macro_avg, k_macro_scatter                        (R12)
// Data layout:
//   M, H  [3][nz][ny][nx] real          W1 [3][hx][nz][ny] complex (y fastest)
//   W2    [3][nkx][nz][Ny] complex, one L2-resident slab of nkx kx-planes
//   K     [6][hx][kpz][kpitch] real, ky' fastest, packed over ky' = min(ky, Ny-ky), kz' likewise
#pragma once
#include "fft_core.cuh"

namespace demag {

struct Geo {
    int nx, ny, nz;        // mesh
    int Nx, Ny, Nz;        // padded sizes
    int hx;                // Nx/2 + 1 (1 if Nx == 1)
    int lLc, lNy, lNz;     // log2(Nx/2), log2(Ny), log2(Nz)
    int kpy, kpz, kpitch;  // packed kernel extents along y, z and the row pitch (elements)
};


// ------------------------------------------------------------------------------------------ K1
// tile = R consecutive y rows of one (component, z); smem s[Lc][R], Lc = Nx/2.
template <typename T>
__global__ void __launch_bounds__(512) k_x_r2c(Geo g, int R, const T* __restrict__ M,
                                               typename cx_of<T>::type* __restrict__ W1,
                                               const typename cx_of<T>::type* __restrict__ twx)
{
    using C = typename cx_of<T>::type;
    constexpr int RB = cx_of<T>::ROWBITS;
    C* s = reinterpret_cast<C*>(demag_smem);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int tilesY = g.ny / R;
    const int ty = blockIdx.x % tilesY;
    const int cz = blockIdx.x / tilesY;            // c*nz + z
    const int y0 = ty * R;
    const int Lc = 1 << g.lLc;
    const int nin = g.nx >> 1;                     // complex pairs holding data per row
    const size_t rowbase = ((size_t)cz * g.ny + y0) * g.nx;
    const int lnin = 31 - __clz(nin);
    for (int idx = tid; idx < R * Lc; idx += nthr) {
        const int b = idx >> g.lLc, m = idx & (Lc - 1);
        C v = cmake<C>((T)0, (T)0);
        if (m < nin) v = *reinterpret_cast<const C*>(M + rowbase + (size_t)b * g.nx + 2 * m);
        s[swz<RB>(m * R + b)] = v;
    }
    (void)lnin;
    __syncthreads();
    fft_tile<T, false>(s, g.lLc, R, twx, 1, tid, nthr);
    const int c = cz / g.nz, z = cz - c * g.nz;
    const size_t plane = (size_t)g.nz * g.ny;
    C* out = W1 + ((size_t)c * g.hx * g.nz + z) * g.ny + y0;
    const bool pow2R = (R & (R - 1)) == 0; const int lR = 31 - __clz(R);
    for (int idx = tid; idx < R * g.hx; idx += nthr) {
        int k, b;
        if (pow2R) { k = idx >> lR; b = idx & (R - 1); } else { k = idx / R; b = idx - k * R; }
        const C Zk = s[swz<RB>(pos_of_freq(k & (Lc - 1), g.lLc) * R + b)];
        const C Zm = s[swz<RB>(pos_of_freq((Lc - k) & (Lc - 1), g.lLc) * R + b)];
        const C E = cmake<C>((T)0.5 * (Zk.x + Zm.x), (T)0.5 * (Zk.y - Zm.y));
        const C D = cmake<C>(Zk.x - Zm.x, Zk.y + Zm.y);
        const C t = cmul(D, __ldg(twx + k));
        out[(size_t)k * plane + b] = cmake<C>(E.x + (T)0.5 * t.y, E.y - (T)0.5 * t.x);
    }
}

// Nx == 1 (nx == 1): the x transform is the identity; W1[c][0][z][y] = M[c][z][y][0].
template <typename T>
__global__ void k_x_copy_fwd(size_t n, const T* __restrict__ M, typename cx_of<T>::type* __restrict__ W1)
{
    using C = typename cx_of<T>::type;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        W1[i] = cmake<C>(M[i], (T)0);
}
template <typename T>
__global__ void k_x_copy_inv(size_t n, const typename cx_of<T>::type* __restrict__ W1, T* __restrict__ H)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        H[i] = W1[i].x;
}

// ------------------------------------------------------------------------------------------ K5
template <typename T>
__global__ void __launch_bounds__(512) k_x_c2r(Geo g, int R, const typename cx_of<T>::type* __restrict__ W1,
                                               T* __restrict__ H,
                                               const typename cx_of<T>::type* __restrict__ twx)
{
    using C = typename cx_of<T>::type;
    constexpr int RB = cx_of<T>::ROWBITS;
    C* s = reinterpret_cast<C*>(demag_smem);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int tilesY = g.ny / R;
    const int ty = blockIdx.x % tilesY;
    const int cz = blockIdx.x / tilesY;
    const int y0 = ty * R;
    const int Lc = 1 << g.lLc;
    const int c = cz / g.nz, z = cz - c * g.nz;
    const size_t plane = (size_t)g.nz * g.ny;
    const C* in = W1 + ((size_t)c * g.hx * g.nz + z) * g.ny + y0;
    const bool pow2R = (R & (R - 1)) == 0; const int lR = 31 - __clz(R);
    for (int idx = tid; idx < R * Lc; idx += nthr) {
        int k, b;
        if (pow2R) { k = idx >> lR; b = idx & (R - 1); } else { k = idx / R; b = idx - k * R; }
        const C Xk = in[(size_t)k * plane + b];
        const C Xm = in[(size_t)(Lc - k) * plane + b];
        const C A = cmake<C>(Xk.x + Xm.x, Xk.y - Xm.y);          // Xk + conj(Xm)
        const C D = cmake<C>(Xk.x - Xm.x, Xk.y + Xm.y);          // Xk - conj(Xm)
        const C u = cmulc(D, __ldg(twx + k));                    // conj(w^k) D
        s[swz<RB>(pos_of_freq(k, g.lLc) * R + b)] = cmake<C>(A.x - u.y, A.y + u.x);   // A + i u
    }
    __syncthreads();
    fft_tile<T, true>(s, g.lLc, R, twx, 1, tid, nthr);
    const int nout = g.nx >> 1;
    const int lno = 31 - __clz(nout);
    const size_t rowbase = ((size_t)cz * g.ny + y0) * g.nx;
    for (int idx = tid; idx < R * nout; idx += nthr) {
        const int b = idx >> lno, m = idx & (nout - 1);
        *reinterpret_cast<C*>(H + rowbase + (size_t)b * g.nx + 2 * m) = s[swz<RB>(m * R + b)];
    }
}

// ------------------------------------------------------------------------------------------ K2 / K4
// lines l = (c*nkx + kxl)*nz + z of the slab [kx0, kx0+nkx); tile = B consecutive lines; smem s[Ny][B].
template <typename T>
__global__ void __launch_bounds__(512) k_y_fwd(Geo g, int B, int kx0, int nkx,
                                               const typename cx_of<T>::type* __restrict__ W1,
                                               typename cx_of<T>::type* __restrict__ W2,
                                               const typename cx_of<T>::type* __restrict__ twy)
{
    using C = typename cx_of<T>::type;
    constexpr int RB = cx_of<T>::ROWBITS;
    C* s = reinterpret_cast<C*>(demag_smem);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int nlines = 3 * nkx * g.nz;
    const int l0 = blockIdx.x * B;
    const int lny = 31 - __clz(g.ny);
    for (int idx = tid; idx < (B << g.lNy); idx += nthr) {
        const int b = idx >> g.lNy, p = idx & (g.Ny - 1);
        const int l = l0 + b;
        C v = cmake<C>((T)0, (T)0);
        if (p < g.ny && l < nlines) {
            const int z = l % g.nz, ck = l / g.nz, kxl = ck % nkx, c = ck / nkx;
            v = W1[(((size_t)c * g.hx + kx0 + kxl) * g.nz + z) * g.ny + p];
        }
        s[swz<RB>(p * B + b)] = v;
    }
    (void)lny;
    __syncthreads();
    fft_tile<T, false>(s, g.lNy, B, twy, 0, tid, nthr);
    for (int idx = tid; idx < (B << g.lNy); idx += nthr) {
        const int b = idx >> g.lNy, ky = idx & (g.Ny - 1);
        const int l = l0 + b;
        if (l < nlines) W2[(size_t)l * g.Ny + ky] = s[swz<RB>(pos_of_freq(ky, g.lNy) * B + b)];
    }
}

template <typename T>
__global__ void __launch_bounds__(512) k_y_inv(Geo g, int B, int kx0, int nkx,
                                               const typename cx_of<T>::type* __restrict__ W2,
                                               typename cx_of<T>::type* __restrict__ W1,
                                               const typename cx_of<T>::type* __restrict__ twy)
{
    using C = typename cx_of<T>::type;
    constexpr int RB = cx_of<T>::ROWBITS;
    C* s = reinterpret_cast<C*>(demag_smem);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int nlines = 3 * nkx * g.nz;
    const int l0 = blockIdx.x * B;
    for (int idx = tid; idx < (B << g.lNy); idx += nthr) {
        const int b = idx >> g.lNy, ky = idx & (g.Ny - 1);
        const int l = l0 + b;
        C v = cmake<C>((T)0, (T)0);
        if (l < nlines) v = W2[(size_t)l * g.Ny + ky];
        s[swz<RB>(pos_of_freq(ky, g.lNy) * B + b)] = v;
    }
    __syncthreads();
    fft_tile<T, true>(s, g.lNy, B, twy, 0, tid, nthr);
    const int lny = 31 - __clz(g.ny);
    for (int idx = tid; idx < (B << lny); idx += nthr) {
        const int b = idx >> lny, p = idx & (g.ny - 1);
        const int l = l0 + b;
        if (l < nlines) {
            const int z = l % g.nz, ck = l / g.nz, kxl = ck % nkx, c = ck / nkx;
            W1[(((size_t)c * g.hx + kx0 + kxl) * g.nz + z) * g.ny + p] = s[swz<RB>(p * B + b)];
        }
    }
}

// ------------------------------------------------------------------------------------------ K3
// tile = one kx plane x TY consecutive ky x all z x 3 components; smem s[Nz][3*TY].
// H^_a = sum_b K^_ab M^_b, K^ real and symmetric (PAPER.md:322-326 KernelMultiplication;
// :255-256 packed by y/z symmetry; parity signs DESIGN.md R1).  In place on the W2 slab.
template <typename T>
__global__ void __launch_bounds__(512) k_z_mul(Geo g, int TY, int kx0, int nkx,
                                               typename cx_of<T>::type* __restrict__ W2,
                                               const T* __restrict__ K, size_t kcomp_stride,
                                               const typename cx_of<T>::type* __restrict__ twz)
{
    using C = typename cx_of<T>::type;
    constexpr int RB = cx_of<T>::ROWBITS;
    C* s = reinterpret_cast<C*>(demag_smem);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int tilesY = g.Ny / TY;
    const int kyt = blockIdx.x % tilesY, kxl = blockIdx.x / tilesY;
    const int ky0 = kyt * TY;
    const int B = 3 * TY;
    const int lTY = 31 - __clz(TY);
    const size_t cstride = (size_t)nkx * g.nz * g.Ny;                 // component stride in the slab
    C* base = W2 + ((size_t)kxl * g.nz) * g.Ny + ky0;
    for (int idx = tid; idx < 3 * g.Nz * TY; idx += nthr) {
        const int ty = idx & (TY - 1), r = idx >> lTY;
        const int z = r & (g.Nz - 1), c = r >> g.lNz;
        C v = cmake<C>((T)0, (T)0);
        if (z < g.nz) v = base[c * cstride + (size_t)z * g.Ny + ty];
        s[swz<RB>(z * B + c * TY + ty)] = v;
    }
    __syncthreads();
    fft_tile<T, false>(s, g.lNz, B, twz, 0, tid, nthr);
    const int kx = kx0 + kxl;
    for (int idx = tid; idx < g.Nz * TY; idx += nthr) {
        const int ty = idx & (TY - 1), p = idx >> lTY;
        const int kz = freq_of_pos(p, g.lNz);
        const int ky = ky0 + ty;
        const bool my = (2 * ky > g.Ny), mz = (2 * kz > g.Nz);
        const int kyp = my ? g.Ny - ky : ky, kzp = mz ? g.Nz - kz : kz;
        const T sy = my ? (T)-1 : (T)1, sz = mz ? (T)-1 : (T)1;
        const size_t ko = ((size_t)kx * g.kpz + kzp) * g.kpitch + kyp;
        const T kxx = __ldg(K + ko), kyy = __ldg(K + kcomp_stride + ko), kzz = __ldg(K + 2 * kcomp_stride + ko);
        const T kxy = sy * __ldg(K + 3 * kcomp_stride + ko);
        const T kxz = sz * __ldg(K + 4 * kcomp_stride + ko);
        const T kyz = sy * sz * __ldg(K + 5 * kcomp_stride + ko);
        const int a0 = swz<RB>(p * B + ty), a1 = swz<RB>(p * B + TY + ty), a2 = swz<RB>(p * B + 2 * TY + ty);
        const C mx = s[a0], my_ = s[a1], mz_ = s[a2];
        s[a0] = cmake<C>(kxx * mx.x + kxy * my_.x + kxz * mz_.x, kxx * mx.y + kxy * my_.y + kxz * mz_.y);
        s[a1] = cmake<C>(kxy * mx.x + kyy * my_.x + kyz * mz_.x, kxy * mx.y + kyy * my_.y + kyz * mz_.y);
        s[a2] = cmake<C>(kxz * mx.x + kyz * my_.x + kzz * mz_.x, kxz * mx.y + kyz * my_.y + kzz * mz_.y);
    }
    __syncthreads();
    fft_tile<T, true>(s, g.lNz, B, twz, 0, tid, nthr);
    const int lnz = 31 - __clz(g.nz);
    for (int idx = tid; idx < ((3 * TY) << lnz); idx += nthr) {
        const int ty = idx & (TY - 1), r = idx >> lTY;
        const int z = r & (g.nz - 1), c = r >> lnz;
        base[c * cstride + (size_t)z * g.Ny + ty] = s[swz<RB>(z * B + c * TY + ty)];
    }
}

// ------------------------------------------------------------------------------------------ energy
// E += -(mu0/2) V sum M.H over this block's cells (fp64 accumulation; R12).
template <typename T>
__global__ void __launch_bounds__(256) k_energy(size_t n3, const T* __restrict__ M, const T* __restrict__ H,
                                                double scale, double* __restrict__ E)
{
    double acc = 0.0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n3; i += (size_t)gridDim.x * blockDim.x)
        acc += (double)M[i] * (double)H[i];
    __shared__ double red[8];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x < 8) {
        acc = red[threadIdx.x];
        for (int o = 4; o > 0; o >>= 1) acc += __shfl_down_sync(0xffu, acc, o);
        if (threadIdx.x == 0) atomicAdd(E, acc * scale);
    }
}

// ------------------------------------------------------------------------------------------ atomistic
// Eq. (9): M_cell = f * sum of the cx*cy*cz unit spins of the cell, f = mu_B mu_s/(c a^3).
template <typename T>
__global__ void __launch_bounds__(256) k_macro_avg(int nx, int ny, int nz, int cx, int cy, int cz,
                                                   const T* __restrict__ S, T* __restrict__ M, double f)
{
    const size_t ncell = (size_t)nx * ny * nz;
    const size_t Lx = (size_t)nx * cx, Ly = (size_t)ny * cy, Lz = (size_t)nz * cz;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < 3 * ncell; i += (size_t)gridDim.x * blockDim.x) {
        const size_t c = i / ncell, cell = i - c * ncell;
        const int X = (int)(cell % nx), Y = (int)((cell / nx) % ny), Z = (int)(cell / ((size_t)nx * ny));
        const T* p = S + ((c * Lz + (size_t)Z * cz) * Ly + (size_t)Y * cy) * Lx + (size_t)X * cx;
        double acc = 0.0;
        for (int dz = 0; dz < cz; ++dz)
            for (int dy = 0; dy < cy; ++dy) {
                const T* q = p + ((size_t)dz * Ly + dy) * Lx;
                if (cx == 4 && sizeof(T) == 4) {
                    const float4 v = *reinterpret_cast<const float4*>(q);
                    acc += ((double)v.x + (double)v.y) + ((double)v.z + (double)v.w);
                } else {
                    for (int dx = 0; dx < cx; ++dx) acc += (double)q[dx];
                }
            }
        M[i] = (T)(acc * f);
    }
}

// the cell field is applied equally to all spins of the cell (copy; optional accumulate).
template <typename T>
__global__ void __launch_bounds__(256) k_macro_scatter(int nx, int ny, int nz, int cx, int cy, int cz,
                                                       const T* __restrict__ H, T* __restrict__ Hs, int accumulate)
{
    const size_t Lx = (size_t)nx * cx, Ly = (size_t)ny * cy, Lz = (size_t)nz * cz;
    const size_t nspin = Lx * Ly * Lz;
    const size_t ncell = (size_t)nx * ny * nz;
    if (cx == 4 && sizeof(T) == 4) {
        const size_t nq = 3 * nspin / 4;
        for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < nq; i += (size_t)gridDim.x * blockDim.x) {
            const size_t e = i * 4;
            const size_t c = e / nspin, r = e - c * nspin;
            const size_t x = r % Lx, y = (r / Lx) % Ly, z = r / (Lx * Ly);
            const float h = (float)H[c * ncell + ((z / cz) * ny + (y / cy)) * nx + x / 4];
            float4* dst = reinterpret_cast<float4*>(Hs) + i;
            float4 v = make_float4(h, h, h, h);
            if (accumulate) { const float4 o = *dst; v.x += o.x; v.y += o.y; v.z += o.z; v.w += o.w; }
            *dst = v;
        }
    } else {
        for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < 3 * nspin; e += (size_t)gridDim.x * blockDim.x) {
            const size_t c = e / nspin, r = e - c * nspin;
            const size_t x = r % Lx, y = (r / Lx) % Ly, z = r / (Lx * Ly);
            const T h = H[c * ncell + ((z / cz) * ny + (y / cy)) * nx + x / cx];
            Hs[e] = accumulate ? Hs[e] + h : h;
        }
    }
}

}  // namespace demag
