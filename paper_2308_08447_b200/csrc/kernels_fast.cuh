// kernels_fast.cuh -- x and y stages for transform lengths >= 16 with >= 2 lines per tile.
// Same mathematics as the generic kernels of kernels.cuh; the difference is data movement:
//   * the first forward pass reads global memory directly (zero padding = the upper half of the
//     butterfly inputs is never loaded) and the last inverse pass writes global memory directly (crop =
//     the upper half of its outputs is never stored): no separate load / store sweep over the tile;
//   * tiles are s[p][pitch] with an odd pitch: a half warp that walks p at fixed line (the global-memory
//     side, coalesced along the line) and one that walks the lines at fixed p (the butterfly side) are
//     both bank-conflict free, without an address swizzle;
//   * the y spectrum stays in the digit-reversed order the forward passes leave it in (W2 "position
//     order"); the kernel spectrum is stored in the same order at plan time, so nothing is permuted.
#pragma once
#include "fft_core.cuh"

namespace demag {

// first forward pass: radix 8, stride S0 = L/8, inputs through ld(b, p); threads walk p fastest
template <typename T, bool HALF, typename LD>
__device__ __forceinline__ void pass_first_fwd(typename cx_of<T>::type* s, int lL, int B, int pitch,
                                               const typename cx_of<T>::type* __restrict__ tw, int lt,
                                               int tid, int nthr, LD ld)
{
    using C = typename cx_of<T>::type;
    const int ls0 = lL - 3, S0 = 1 << ls0, nb = B << ls0;
    for (int t = tid; t < nb; t += nthr) {
        const int i = t & (S0 - 1), b = t >> ls0;
        C a[8];
#pragma unroll
        for (int r = 0; r < (HALF ? 4 : 8); ++r) a[r] = ld(b, i + r * S0);
        dft8<false, HALF>(a);
        twiddle<3, false, false>(a, tw, i << lt);
        C* d = s + i * pitch + b;
        const int st = S0 * pitch;
#pragma unroll
        for (int r = 0; r < 8; ++r) d[r * st] = a[r];
    }
}

// last inverse pass: radix 8, stride S0 = L/8, outputs r < nout through st(b, p, v); threads walk p fastest
template <typename T, typename ST>
__device__ __forceinline__ void pass_last_inv(typename cx_of<T>::type* s, int lL, int B, int pitch,
                                              const typename cx_of<T>::type* __restrict__ tw, int lt,
                                              int tid, int nthr, bool half_out, ST stf)
{
    using C = typename cx_of<T>::type;
    const int ls0 = lL - 3, S0 = 1 << ls0, nb = B << ls0;
    for (int t = tid; t < nb; t += nthr) {
        const int i = t & (S0 - 1), b = t >> ls0;
        C a[8];
        const C* d = s + i * pitch + b;
        const int st = S0 * pitch;
#pragma unroll
        for (int r = 0; r < 8; ++r) a[r] = d[r * st];
        twiddle<3, true, false>(a, tw, i << lt);
        dft8<true, false>(a);
#pragma unroll
        for (int r = 0; r < 8; ++r) if (r < 4 || !half_out) stf(b, i + r * S0, a[r]);
    }
}

// the passes between: forward = all but the first, inverse = all but the last; in place, lines fastest
template <typename T, bool INV>
__device__ __forceinline__ void fft_mid(typename cx_of<T>::type* s, int lL, int B, int pitch,
                                        const typename cx_of<T>::type* __restrict__ tw, int lt, int tid, int nthr)
{
    const int n8 = lL / 3, rem = lL % 3;
    if (!INV) {
        for (int k = 1; k < n8; ++k) { fft_pass<T, 3, false, false>(s, lL, lL - 3 * (k + 1), B, pitch, tw, lt, tid, nthr); __syncthreads(); }
        if (rem == 2) { fft_pass<T, 2, false, false>(s, lL, 0, B, pitch, tw, lt, tid, nthr); __syncthreads(); }
        else if (rem == 1) { fft_pass<T, 1, false, false>(s, lL, 0, B, pitch, tw, lt, tid, nthr); __syncthreads(); }
    } else {
        if (rem == 2) { fft_pass<T, 2, true, false>(s, lL, 0, B, pitch, tw, lt, tid, nthr); __syncthreads(); }
        else if (rem == 1) { fft_pass<T, 1, true, false>(s, lL, 0, B, pitch, tw, lt, tid, nthr); __syncthreads(); }
        for (int k = n8 - 1; k >= 1; --k) { fft_pass<T, 3, true, false>(s, lL, lL - 3 * (k + 1), B, pitch, tw, lt, tid, nthr); __syncthreads(); }
    }
}

// ------------------------------------------------------------------------------------------ K1 fast
template <typename T>
__global__ void __launch_bounds__(512) k_x_r2c_f(Geo g, int R, int pitch, const T* __restrict__ M,
                                                 typename cx_of<T>::type* __restrict__ W1,
                                                 const typename cx_of<T>::type* __restrict__ twx)
{
    using C = typename cx_of<T>::type;
    C* s = reinterpret_cast<C*>(demag_smem);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int tilesY = g.ny / R;
    const int ty = blockIdx.x % tilesY;
    const int cz = blockIdx.x / tilesY;            // c*nz + z
    const int y0 = ty * R;
    const int Lc = 1 << g.lLc;
    const T* rows = M + ((size_t)cz * g.ny + y0) * g.nx;
    const int nx = g.nx;
    auto ld = [&](int b, int m) { return *reinterpret_cast<const C*>(rows + (size_t)b * nx + 2 * m); };
    if (g.Nx != g.nx) pass_first_fwd<T, true>(s, g.lLc, R, pitch, twx, 1, tid, nthr, ld);
    else pass_first_fwd<T, false>(s, g.lLc, R, pitch, twx, 1, tid, nthr, ld);
    __syncthreads();
    fft_mid<T, false>(s, g.lLc, R, pitch, twx, 1, tid, nthr);
    const int c = cz / g.nz, z = cz - c * g.nz;
    const size_t plane = (size_t)g.nz * g.ny;
    C* out = W1 + ((size_t)c * g.hx * g.nz + z) * g.ny + y0;
    const int lR = 31 - __clz(R);                  // R is a power of two
    for (int idx = tid; idx < R * g.hx; idx += nthr) {
        const int k = idx >> lR, b = idx & (R - 1);
        const C Zk = s[pos_of_freq(k & (Lc - 1), g.lLc) * pitch + b];
        const C Zm = s[pos_of_freq((Lc - k) & (Lc - 1), g.lLc) * pitch + b];
        const C E = cmake<C>((T)0.5 * (Zk.x + Zm.x), (T)0.5 * (Zk.y - Zm.y));
        const C D = cmake<C>(Zk.x - Zm.x, Zk.y + Zm.y);
        const C t = cmul(D, __ldg(twx + k));
        out[(size_t)k * plane + b] = cmake<C>(E.x + (T)0.5 * t.y, E.y - (T)0.5 * t.x);
    }
}

// ------------------------------------------------------------------------------------------ K5 fast
template <typename T>
__global__ void __launch_bounds__(512) k_x_c2r_f(Geo g, int R, int pitch, const typename cx_of<T>::type* __restrict__ W1,
                                                 T* __restrict__ H,
                                                 const typename cx_of<T>::type* __restrict__ twx)
{
    using C = typename cx_of<T>::type;
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
    const int lR = 31 - __clz(R);
    for (int idx = tid; idx < R * Lc; idx += nthr) {
        const int k = idx >> lR, b = idx & (R - 1);
        const C Xk = in[(size_t)k * plane + b];
        const C Xm = in[(size_t)(Lc - k) * plane + b];
        const C A = cmake<C>(Xk.x + Xm.x, Xk.y - Xm.y);          // Xk + conj(Xm)
        const C D = cmake<C>(Xk.x - Xm.x, Xk.y + Xm.y);          // Xk - conj(Xm)
        const C u = cmulc(D, __ldg(twx + k));                    // conj(w^k) D
        s[pos_of_freq(k, g.lLc) * pitch + b] = cmake<C>(A.x - u.y, A.y + u.x);   // A + i u
    }
    __syncthreads();
    fft_mid<T, true>(s, g.lLc, R, pitch, twx, 1, tid, nthr);
    T* rows = H + ((size_t)cz * g.ny + y0) * g.nx;
    const int nx = g.nx;
    const int acc = g.acc;
    auto stf = [&](int b, int m, C v) {
        C* d = reinterpret_cast<C*>(rows + (size_t)b * nx + 2 * m);
        if (acc) { const C o = *d; v.x += o.x; v.y += o.y; }
        *d = v;
    };
    pass_last_inv<T>(s, g.lLc, R, pitch, twx, 1, tid, nthr, g.Nx != g.nx, stf);
}

// ------------------------------------------------------------------------------------------ K2 / K4 fast
// lines l = (c*nkx + kxl)*nz + z of the slab [kx0, kx0+nkx); tile = B consecutive lines; smem s[Ny][pitch].
__device__ __forceinline__ size_t w1_line_offset(const Geo& g, int l, int kx0, int nkx)
{
    const int z = l % g.nz, ck = l / g.nz, kxl = ck % nkx, c = ck / nkx;
    return (((size_t)c * g.hx + kx0 + kxl) * g.nz + z) * g.ny;
}

template <typename T>
__global__ void __launch_bounds__(512) k_y_fwd_f(Geo g, int B, int pitch, int kx0, int nkx,
                                                 const typename cx_of<T>::type* __restrict__ W1,
                                                 typename cx_of<T>::type* __restrict__ W2,
                                                 const typename cx_of<T>::type* __restrict__ twy)
{
    using C = typename cx_of<T>::type;
    C* s = reinterpret_cast<C*>(demag_smem);
    __shared__ long long loff[16];
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int nlines = 3 * nkx * g.nz;
    const int l0 = blockIdx.x * B;
    if (tid < B) loff[tid] = (l0 + tid < nlines) ? (long long)w1_line_offset(g, l0 + tid, kx0, nkx) : -1;
    __syncthreads();
    auto ld = [&](int b, int p) { const long long o = loff[b]; return o >= 0 ? W1[o + p] : cmake<C>((T)0, (T)0); };
    if (g.Ny != g.ny) pass_first_fwd<T, true>(s, g.lNy, B, pitch, twy, 0, tid, nthr, ld);
    else pass_first_fwd<T, false>(s, g.lNy, B, pitch, twy, 0, tid, nthr, ld);
    __syncthreads();
    fft_mid<T, false>(s, g.lNy, B, pitch, twy, 0, tid, nthr);
    // position-order store: W2[l][p] = s[p][b], threads walk p fastest (coalesced, conflict free)
    C* dst = W2 + (size_t)l0 * g.Ny;
    const int nvalid = min(B, nlines - l0);
    for (int idx = tid; idx < (nvalid << g.lNy); idx += nthr) {
        const int b = idx >> g.lNy, p = idx & (g.Ny - 1);
        dst[idx] = s[p * pitch + b];
    }
}

template <typename T>
__global__ void __launch_bounds__(512) k_y_inv_f(Geo g, int B, int pitch, int kx0, int nkx,
                                                 const typename cx_of<T>::type* __restrict__ W2,
                                                 typename cx_of<T>::type* __restrict__ W1,
                                                 const typename cx_of<T>::type* __restrict__ twy)
{
    using C = typename cx_of<T>::type;
    C* s = reinterpret_cast<C*>(demag_smem);
    __shared__ long long loff[16];
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int nlines = 3 * nkx * g.nz;
    const int l0 = blockIdx.x * B;
    if (tid < B) loff[tid] = (l0 + tid < nlines) ? (long long)w1_line_offset(g, l0 + tid, kx0, nkx) : -1;
    const C* src = W2 + (size_t)l0 * g.Ny;
    const int nvalid = min(B, nlines - l0);
    for (int idx = tid; idx < (B << g.lNy); idx += nthr) {
        const int b = idx >> g.lNy, p = idx & (g.Ny - 1);
        s[p * pitch + b] = b < nvalid ? src[idx] : cmake<C>((T)0, (T)0);
    }
    __syncthreads();
    fft_mid<T, true>(s, g.lNy, B, pitch, twy, 0, tid, nthr);
    auto stf = [&](int b, int p, C v) { const long long o = loff[b]; if (o >= 0) W1[o + p] = v; };
    pass_last_inv<T>(s, g.lNy, B, pitch, twy, 0, tid, nthr, g.Ny != g.ny, stf);
}

}  // namespace demag
