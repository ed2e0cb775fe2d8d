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
//   K     [6][hx][kpz][Ny] real: z packed over kz' = min(kz, Nz-kz); y unpacked, in W2's position order
#pragma once
#include "fft_core.cuh"

namespace demag {

struct Geo {
    int nx, ny, nz;        // mesh
    int Nx, Ny, Nz;        // padded sizes
    int hx;                // Nx/2 + 1 (1 if Nx == 1)
    int lLc, lNy, lNz;     // log2(Nx/2), log2(Ny), log2(Nz)
    int kpy, kpz, kpitch;  // packed kernel extents along y, z and the row pitch (elements)
    int acc;               // x C2R: 0 = overwrite H, 1 = add into H (demag_apply_add)
};


// ------------------------------------------------------------------------------------------ K1
// tile = R consecutive y rows of one (component, z); smem s[Lc][R], Lc = Nx/2.
template <typename T, bool SWZ>
__global__ void __launch_bounds__(512) k_x_r2c(Geo g, int R, int pitch, const T* __restrict__ M,
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
        s[taddr<SWZ, RB>(m * pitch + b)] = v;
    }
    (void)lnin;
    __syncthreads();
    fft_tile<T, false, SWZ>(s, g.lLc, R, pitch, twx, 1, tid, nthr);
    const int c = cz / g.nz, z = cz - c * g.nz;
    const size_t plane = (size_t)g.nz * g.ny;
    C* out = W1 + ((size_t)c * g.hx * g.nz + z) * g.ny + y0;
    const bool pow2R = (R & (R - 1)) == 0; const int lR = 31 - __clz(R);
    for (int idx = tid; idx < R * g.hx; idx += nthr) {
        int k, b;
        if (pow2R) { k = idx >> lR; b = idx & (R - 1); } else { k = idx / R; b = idx - k * R; }
        const C Zk = s[taddr<SWZ, RB>(pos_of_freq(k & (Lc - 1), g.lLc) * pitch + b)];
        const C Zm = s[taddr<SWZ, RB>(pos_of_freq((Lc - k) & (Lc - 1), g.lLc) * pitch + b)];
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
__global__ void k_x_copy_inv(size_t n, const typename cx_of<T>::type* __restrict__ W1, T* __restrict__ H, int acc)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        H[i] = acc ? H[i] + W1[i].x : W1[i].x;
}

// ------------------------------------------------------------------------------------------ K5
template <typename T, bool SWZ>
__global__ void __launch_bounds__(512) k_x_c2r(Geo g, int R, int pitch, const typename cx_of<T>::type* __restrict__ W1,
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
        s[taddr<SWZ, RB>(pos_of_freq(k, g.lLc) * pitch + b)] = cmake<C>(A.x - u.y, A.y + u.x);   // A + i u
    }
    __syncthreads();
    fft_tile<T, true, SWZ>(s, g.lLc, R, pitch, twx, 1, tid, nthr);
    const int nout = g.nx >> 1;
    const int lno = 31 - __clz(nout);
    const size_t rowbase = ((size_t)cz * g.ny + y0) * g.nx;
    for (int idx = tid; idx < R * nout; idx += nthr) {
        const int b = idx >> lno, m = idx & (nout - 1);
        C v = s[taddr<SWZ, RB>(m * pitch + b)];
        C* d = reinterpret_cast<C*>(H + rowbase + (size_t)b * g.nx + 2 * m);
        if (g.acc) { const C o = *d; v.x += o.x; v.y += o.y; }
        *d = v;
    }
}

// ------------------------------------------------------------------------------------------ K2 / K4
// lines l = (c*nkx + kxl)*nz + z of the slab [kx0, kx0+nkx); tile = B consecutive lines; smem s[Ny][B].
template <typename T, bool SWZ>
__global__ void __launch_bounds__(512) k_y_fwd(Geo g, int B, int pitch, int kx0, int nkx,
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
        s[taddr<SWZ, RB>(p * pitch + b)] = v;
    }
    (void)lny;
    __syncthreads();
    fft_tile<T, false, SWZ>(s, g.lNy, B, pitch, twy, 0, tid, nthr);
    for (int idx = tid; idx < (B << g.lNy); idx += nthr) {
        const int b = idx >> g.lNy, ky = idx & (g.Ny - 1);
        const int l = l0 + b;
        if (l < nlines) W2[(size_t)l * g.Ny + ky] = s[taddr<SWZ, RB>(ky * pitch + b)];   // W2 keeps position (digit-reversed) order
    }
}

template <typename T, bool SWZ>
__global__ void __launch_bounds__(512) k_y_inv(Geo g, int B, int pitch, int kx0, int nkx,
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
        s[taddr<SWZ, RB>(ky * pitch + b)] = v;
    }
    __syncthreads();
    fft_tile<T, true, SWZ>(s, g.lNy, B, pitch, twy, 0, tid, nthr);
    const int lny = 31 - __clz(g.ny);
    for (int idx = tid; idx < (B << lny); idx += nthr) {
        const int b = idx >> lny, p = idx & (g.ny - 1);
        const int l = l0 + b;
        if (l < nlines) {
            const int z = l % g.nz, ck = l / g.nz, kxl = ck % nkx, c = ck / nkx;
            W1[(((size_t)c * g.hx + kx0 + kxl) * g.nz + z) * g.ny + p] = s[taddr<SWZ, RB>(p * pitch + b)];
        }
    }
}

// ------------------------------------------------------------------------------------------ K3
// z FFT . kernel multiplication . z IFFT "in the same routine".
// tile = one kx plane x TY consecutive ky x all z x 3 components; smem s[Nz][3*TY] (batch fastest, so
// every shared-memory access of a half warp is 16 consecutive slots: conflict free, no swizzle).
//   first forward pass   reads W2 straight from global (only z < nz: the zero padding is synthesised)
//   fused middle stage   last forward pass + H^_a = sum_b K^_ab M^_b + first inverse pass, in registers
//   last inverse pass    writes z < nz straight back to W2 (the crop)
// H^_a = sum_b K^_ab M^_b, K^ real and symmetric (PAPER.md:322-326 KernelMultiplication; :255-256 packed
// by y/z symmetry; parity signs DESIGN.md R1).  In place on the W2 slab.
template <typename T>
struct KernelVals { T xx, yy, zz, xy, xz, yz; };

// K is stored [comp][kx][kz'][py]: z packed over kz' = min(kz, Nz-kz) (sign applied here), y unpacked in the
// position order of W2 with its parity sign already folded in at plan time.
template <typename T>
__device__ __forceinline__ KernelVals<T> load_kernel(const Geo& g, const T* __restrict__ K, size_t kcs, int kx, int py, int kz)
{
    const bool mz = (2 * kz > g.Nz);
    const int kzp = mz ? g.Nz - kz : kz;
    const size_t ko = ((size_t)kx * g.kpz + kzp) * g.kpitch + py;
    KernelVals<T> v;
    v.xx = __ldg(K + ko); v.yy = __ldg(K + kcs + ko); v.zz = __ldg(K + 2 * kcs + ko);
    v.xy = __ldg(K + 3 * kcs + ko);
    const T xz = __ldg(K + 4 * kcs + ko), yz = __ldg(K + 5 * kcs + ko);
    v.xz = mz ? -xz : xz; v.yz = mz ? -yz : yz;
    return v;
}

template <typename C, typename T>
__device__ __forceinline__ void apply_kernel(const KernelVals<T>& k, C& mx, C& my, C& mz)
{
    const C kxx = cmake<C>(k.xx, k.xx), kyy = cmake<C>(k.yy, k.yy), kzz = cmake<C>(k.zz, k.zz);
    const C kxy = cmake<C>(k.xy, k.xy), kxz = cmake<C>(k.xz, k.xz), kyz = cmake<C>(k.yz, k.yz);
    const C hx = p_fma(kxz, mz, p_fma(kxy, my, p_mul(kxx, mx)));
    const C hy = p_fma(kyz, mz, p_fma(kyy, my, p_mul(kxy, mx)));
    const C hz = p_fma(kzz, mz, p_fma(kyz, my, p_mul(kxz, mx)));
    mx = hx; my = hy; mz = hz;
}

// fused middle stage on the tile: radix 2^LR, stride 1
template <typename T, int LR>
__device__ __forceinline__ void k3_fused(const Geo& g, typename cx_of<T>::type* s, int TY, int kx, int ky0,
                                         const T* __restrict__ K, size_t kcs, int tid, int nthr)
{
    using C = typename cx_of<T>::type;
    constexpr int R = 1 << LR;
    const int B = 3 * TY;
    const int ty = tid % TY, i0 = tid / TY, istep = nthr / TY;
    const int nbf = g.Nz >> LR;
    for (int i = i0; i < nbf; i += istep) {
        const int p0 = i << LR;
        C a[3][R];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
#pragma unroll
            for (int m = 0; m < R; ++m) a[c][m] = s[(p0 + m) * B + c * TY + ty];
            dftR<LR, false, false>(a[c]);
        }
        const int kb = freq_of_pos(p0, g.lNz);
#pragma unroll
        for (int m = 0; m < R; ++m) {
            const KernelVals<T> kv = load_kernel<T>(g, K, kcs, kx, ky0 + ty, kb + m * (g.Nz >> LR));
            apply_kernel(kv, a[0][m], a[1][m], a[2][m]);
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            dftR<LR, true, false>(a[c]);
#pragma unroll
            for (int m = 0; m < R; ++m) s[(p0 + m) * B + c * TY + ty] = a[c][m];
        }
    }
}

// whole z transform in one radix-2^LR butterfly per (ky, component): Nz <= 8, no shared memory
template <typename T, int LR>
__device__ __forceinline__ void k3_single(const Geo& g, typename cx_of<T>::type* base, size_t cstride, int kx, int ky,
                                          const T* __restrict__ K, size_t kcs)
{
    using C = typename cx_of<T>::type;
    constexpr int R = 1 << LR;
    C a[3][R];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
#pragma unroll
        for (int r = 0; r < R; ++r) a[c][r] = (r < g.nz) ? base[c * cstride + (size_t)r * g.Ny] : cmake<C>((T)0, (T)0);
        dftR<LR, false, false>(a[c]);
    }
#pragma unroll
    for (int m = 0; m < R; ++m) {
        const KernelVals<T> kv = load_kernel<T>(g, K, kcs, kx, ky, m);
        apply_kernel(kv, a[0][m], a[1][m], a[2][m]);
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        dftR<LR, true, false>(a[c]);
#pragma unroll
        for (int r = 0; r < R; ++r) if (r < g.nz) base[c * cstride + (size_t)r * g.Ny] = a[c][r];
    }
}

// Nz <= 8: one thread per ky column, no shared memory.  grid = nkx * Ny / TY, block >= TY.
template <typename T>
__global__ void __launch_bounds__(128) k_z_small(Geo g, int TY, int kx0, int nkx,
                                                 typename cx_of<T>::type* __restrict__ W2,
                                                 const T* __restrict__ K, size_t kcs)
{
    using C = typename cx_of<T>::type;
    const int tid = threadIdx.x;
    const int tilesY = g.Ny / TY;
    const int kyt = blockIdx.x % tilesY, kxl = blockIdx.x / tilesY;
    const int ky0 = kyt * TY;
    const int kx = kx0 + kxl;
    const size_t cstride = (size_t)nkx * g.nz * g.Ny;
    if (tid >= TY) return;
    C* col = W2 + ((size_t)kxl * g.nz) * g.Ny + ky0 + tid;
    const int lNz = g.lNz;
    if (lNz == 0) k3_single<T, 0>(g, col, cstride, kx, ky0 + tid, K, kcs);
    else if (lNz == 1) k3_single<T, 1>(g, col, cstride, kx, ky0 + tid, K, kcs);
    else if (lNz == 2) k3_single<T, 2>(g, col, cstride, kx, ky0 + tid, K, kcs);
    else k3_single<T, 3>(g, col, cstride, kx, ky0 + tid, K, kcs);
}

// Nz >= 16.  LRF = log2 radix of the fused middle stage = the last pass of the schedule (Nz % 8 -> 1, 2; else 3).
template <typename T, int LRF>
__global__ void __launch_bounds__(512, ((LRF == 3 || sizeof(T) == 8) ? 1 : 2)) k_z_mul(Geo g, int TY, int kx0, int nkx,
                                               typename cx_of<T>::type* __restrict__ W2,
                                               const T* __restrict__ K, size_t kcs,
                                               const typename cx_of<T>::type* __restrict__ twz)
{
    using C = typename cx_of<T>::type;
    C* s = reinterpret_cast<C*>(demag_smem);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int tilesY = g.Ny / TY;
    const int kyt = blockIdx.x % tilesY, kxl = blockIdx.x / tilesY;
    const int ky0 = kyt * TY;
    const int kx = kx0 + kxl;
    const size_t cstride = (size_t)nkx * g.nz * g.Ny;                 // component stride in the slab
    C* base = W2 + ((size_t)kxl * g.nz) * g.Ny + ky0;
    const int lNz = g.lNz;
    const int B = 3 * TY;
    const int n8 = lNz / 3, rem = lNz % 3;
    const int npass = n8 + (rem ? 1 : 0);
    const int b = tid % B, i0 = tid / B, istep = nthr / B;       // nthr is a multiple of B (plan)
    const int c = b / TY, ty = b - c * TY;
    C* gcol = base + c * cstride + ty;
    const bool padded = g.Nz != g.nz;
    const int ls0 = lNz - 3, S0 = 1 << ls0;
    // ---- first forward pass (radix 8, stride Nz/8) straight from global
    for (int i = i0; i < S0; i += istep) {
        C a[8];
        if (padded) {
#pragma unroll
            for (int r = 0; r < 4; ++r) a[r] = gcol[(size_t)(i + r * S0) * g.Ny];
            dft8<false, true>(a);
        } else {
#pragma unroll
            for (int r = 0; r < 8; ++r) a[r] = gcol[(size_t)(i + r * S0) * g.Ny];
            dft8<false, false>(a);
        }
        twiddle<3, false, true>(a, twz, i);
#pragma unroll
        for (int r = 0; r < 8; ++r) s[(i + r * S0) * B + b] = a[r];
    }
    __syncthreads();
    // ---- middle forward passes (all radix 8); the last pass of the schedule is the fused stage
    for (int k = 1; k <= npass - 2; ++k) { fft_pass<T, 3, false, false>(s, lNz, lNz - 3 * (k + 1), B, B, twz, 0, tid, nthr); __syncthreads(); }
    k3_fused<T, LRF>(g, s, TY, kx, ky0, K, kcs, tid, nthr);
    __syncthreads();
    for (int k = npass - 2; k >= 1; --k) { fft_pass<T, 3, true, false>(s, lNz, lNz - 3 * (k + 1), B, B, twz, 0, tid, nthr); __syncthreads(); }
    // ---- last inverse pass (radix 8, stride Nz/8) straight to global, keeping z < nz (the crop)
    for (int i = i0; i < S0; i += istep) {
        C a[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) a[r] = s[(i + r * S0) * B + b];
        twiddle<3, true, true>(a, twz, i);
        dft8<true, false>(a);
        const int nout = padded ? 4 : 8;
#pragma unroll
        for (int r = 0; r < 8; ++r) if (r < nout) gcol[(size_t)(i + r * S0) * g.Ny] = a[r];
    }
}

// ------------------------------------------------------------------------------------------ energy
// E += -(mu0/2) V sum M.H over this block's cells (fp64 accumulation; R12).
// Polynomial extrapolation of the demagnetizing field at a sub-step of the time integrator (DESIGN.md
// R19):  out (+)= sum_k w[k] H_k  over NP previously computed fields, w = the Lagrange weights L_k(t), computed on the
// host in fp64.  One streaming pass: NP reads (+1 when accumulating) and one write per element, 16-byte accesses.
constexpr int kMaxHist = 8;
template <typename T> struct ExtrapArgs { const T* H[kMaxHist]; T w[kMaxHist]; };
template <typename T, int NP>
__global__ void __launch_bounds__(256) k_extrapolate(size_t n, ExtrapArgs<T> a, T* __restrict__ out, int acc)
{
    constexpr int V = 16 / (int)sizeof(T);
    struct alignas(16) Vec { T v[V]; };
    const size_t nvec = n / V;
    const size_t stride = (size_t)gridDim.x * blockDim.x, i0 = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    for (size_t i = i0; i < nvec; i += stride) {
        Vec h[NP];
#pragma unroll
        for (int k = 0; k < NP; ++k) h[k] = reinterpret_cast<const Vec*>(a.H[k])[i];
        Vec r;
        if (acc) r = reinterpret_cast<const Vec*>(out)[i];
        else {
#pragma unroll
            for (int e = 0; e < V; ++e) r.v[e] = (T)0;
        }
#pragma unroll
        for (int k = 0; k < NP; ++k) {
#pragma unroll
            for (int e = 0; e < V; ++e) r.v[e] = fma(a.w[k], h[k].v[e], r.v[e]);
        }
        reinterpret_cast<Vec*>(out)[i] = r;
    }
    for (size_t i = nvec * V + i0; i < n; i += stride) {          // tail (n not a multiple of the vector width)
        T r = acc ? out[i] : (T)0;
#pragma unroll
        for (int k = 0; k < NP; ++k) r = fma(a.w[k], a.H[k][i], r);
        out[i] = r;
    }
}

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

// Fast variants for macrocells of 4 spins along x (one float4 per cell row): 3D grids, no index divisions.
// grid (ceil(nx / 128), ny, 3 nz), block 128: one thread = one cell of one component.
__global__ void __launch_bounds__(128) k_macro_avg_x4(int nx, int cy, int cz, const float* __restrict__ S,
                                                      float* __restrict__ M, double f)
{
    const int X = blockIdx.x * 128 + threadIdx.x;
    if (X >= nx) return;
    const int Y = blockIdx.y, cZ = blockIdx.z;                       // cZ = c * nz + Z
    const size_t Lx = (size_t)nx * 4, Ly = (size_t)gridDim.y * cy;
    const float4* p = reinterpret_cast<const float4*>(S + (((size_t)cZ * cz) * Ly + (size_t)Y * cy) * Lx) + X;
    const size_t rowq = Lx / 4;
    double acc = 0.0;
    for (int dz = 0; dz < cz; ++dz) {
#pragma unroll 4
        for (int dy = 0; dy < cy; ++dy) {
            const float4 v = __ldcs(p + ((size_t)dz * Ly + dy) * rowq);
            acc += (double)((v.x + v.y) + (v.z + v.w));
        }
    }
    M[((size_t)cZ * gridDim.y + Y) * nx + X] = (float)(acc * f);
}
// grid (ceil(nx / 128), ny, 3 nz), block 128: one thread writes the cy*cz float4 rows of its cell.
__global__ void __launch_bounds__(128) k_macro_scatter_x4(int nx, int cy, int cz, const float* __restrict__ H,
                                                          float* __restrict__ Hs, int accumulate)
{
    const int X = blockIdx.x * 128 + threadIdx.x;
    if (X >= nx) return;
    const int Y = blockIdx.y, cZ = blockIdx.z;
    const size_t Lx = (size_t)nx * 4, Ly = (size_t)gridDim.y * cy;
    const float h = H[((size_t)cZ * gridDim.y + Y) * nx + X];
    float4* p = reinterpret_cast<float4*>(Hs + (((size_t)cZ * cz) * Ly + (size_t)Y * cy) * Lx) + X;
    const size_t rowq = Lx / 4;
    for (int dz = 0; dz < cz; ++dz) {
#pragma unroll 4
        for (int dy = 0; dy < cy; ++dy) {
            float4* d = p + ((size_t)dz * Ly + dy) * rowq;
            float4 v = make_float4(h, h, h, h);
            if (accumulate) { const float4 o = *d; v.x += o.x; v.y += o.y; v.z += o.z; v.w += o.w; }
            __stcs(d, v);
        }
    }
}

}  // namespace demag

#include "kernels_fast.cuh"
