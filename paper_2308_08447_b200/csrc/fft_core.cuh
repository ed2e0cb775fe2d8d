// fft_core.cuh -- in-shared-memory batched power-of-two FFT used by every stage of the
// demagnetizing-field convolution ("N and M are first transformed using a FFT";
// Appendix A :296-321 xFFT / yFFT / zFFT).  sm_100a only; no cuFFT.
//
// A tile is a logical array  s[p][b]  of complex numbers, p = 0..L-1 the transform axis, b = 0..B-1
// the batch (independent lines), flattened q = p*B + b and XOR-swizzled so that both unit-stride and
// power-of-two-strided accesses of a half warp fall in distinct banks (no padding bytes).
//
// Forward  = decimation in frequency, in place, natural order in  -> digit-reversed order out.
// Inverse  = decimation in time,      in place, digit-reversed in -> natural order out.
// The convolution never needs the permutation undone in shared memory: the loaders / storers address
// the tile through pos_of_freq().  Neither direction scales; the 1/(Nx Ny Nz) lives in the kernel
// spectrum (R3).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace demag {

extern __shared__ __align__(16) unsigned char demag_smem[];

template <typename T> struct cx_of;
template <> struct cx_of<float>  { using type = float2;  static constexpr int ROWBITS = 4; };
template <> struct cx_of<double> { using type = double2; static constexpr int ROWBITS = 3; };

template <typename C> __device__ __forceinline__ C cmake(decltype(C::x) a, decltype(C::x) b) { C r; r.x = a; r.y = b; return r; }
template <typename C> __device__ __forceinline__ C cadd(C a, C b) { return cmake<C>(a.x + b.x, a.y + b.y); }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { return cmake<C>(a.x - b.x, a.y - b.y); }
template <typename C> __device__ __forceinline__ C cmul(C a, C b) { return cmake<C>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
template <typename C> __device__ __forceinline__ C cmulc(C a, C b) { /* a * conj(b) */ return cmake<C>(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }
template <typename C> __device__ __forceinline__ C cconj(C a) { return cmake<C>(a.x, -a.y); }
// multiply by -i (forward) or +i (inverse)
template <bool INV, typename C> __device__ __forceinline__ C cmul_mi(C a) { return INV ? cmake<C>(-a.y, a.x) : cmake<C>(a.y, -a.x); }

// XOR swizzle of the flattened element index: rows of 2^ROWBITS elements (= 128 bytes), the in-row
// index is XORed with the folded row number.
template <int ROWBITS> __device__ __forceinline__ int swz(int q)
{
    const int r = q >> ROWBITS;
    const int f = (r ^ (r >> ROWBITS) ^ (r >> (2 * ROWBITS)) ^ (r >> (3 * ROWBITS))) & ((1 << ROWBITS) - 1);
    return q ^ f;
}

// Pass schedule for length 2^log2L: radix-8 passes, then one radix-4 or radix-2 pass.
struct Sched {
    int log2L;
    __device__ __host__ __forceinline__ int npass() const { return (log2L + 2) / 3; }
    __device__ __host__ __forceinline__ int lr(int i) const { return (i < log2L / 3) ? 3 : (log2L % 3); }
};

// position (in the digit-reversed tile) that holds frequency k after the forward passes
__device__ __forceinline__ int pos_of_freq(int k, int log2L)
{
    int p = 0, ls = log2L;                       // ls = log2 of the remaining sub-transform size
    const int n8 = log2L / 3, rem = log2L % 3;
    for (int i = 0; i < n8; ++i) { ls -= 3; p += (k & 7) << ls; k >>= 3; }
    if (rem) { p += k & ((1 << rem) - 1); }
    return p;
}
__device__ __forceinline__ int freq_of_pos(int p, int log2L)
{
    int k = 0, ls = log2L, sh = 0;
    const int n8 = log2L / 3, rem = log2L % 3;
    for (int i = 0; i < n8; ++i) { ls -= 3; k += ((p >> ls) & 7) << sh; sh += 3; }
    if (rem) { k += (p & ((1 << rem) - 1)) << sh; }
    return k;
}

// ---- radix butterflies in registers: natural order in, natural order out, unnormalised ------------
template <bool INV, typename C> __device__ __forceinline__ void dft2(C* a)
{
    const C t = a[0]; a[0] = cadd(t, a[1]); a[1] = csub(t, a[1]);
}
template <bool INV, typename C> __device__ __forceinline__ void dft4(C* a)
{
    const C d0 = cadd(a[0], a[2]), d2 = csub(a[0], a[2]);
    const C d1 = cadd(a[1], a[3]), d3 = cmul_mi<INV>(csub(a[1], a[3]));
    a[0] = cadd(d0, d1); a[2] = csub(d0, d1);
    a[1] = cadd(d2, d3); a[3] = csub(d2, d3);
}
template <bool INV, typename C> __device__ __forceinline__ void dft8(C* a)
{
    using T = decltype(C::x);
    const T h = (T)0.70710678118654752440;
    C e[4], o[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) { e[j] = cadd(a[j], a[j + 4]); o[j] = csub(a[j], a[j + 4]); }
    // o[j] *= w8^j   (forward w8 = exp(-i pi/4); inverse conj)
    {
        const C t1 = o[1], t3 = o[3];
        if (!INV) { o[1] = cmake<C>((t1.x + t1.y) * h, (t1.y - t1.x) * h); o[3] = cmake<C>((t3.y - t3.x) * h, -(t3.x + t3.y) * h); }
        else      { o[1] = cmake<C>((t1.x - t1.y) * h, (t1.x + t1.y) * h); o[3] = cmake<C>(-(t3.x + t3.y) * h, (t3.x - t3.y) * h); }
        o[2] = cmul_mi<INV>(o[2]);
    }
    dft4<INV>(e); dft4<INV>(o);
#pragma unroll
    for (int j = 0; j < 4; ++j) { a[2 * j] = e[j]; a[2 * j + 1] = o[j]; }
}
template <int LR, bool INV, typename C> __device__ __forceinline__ void dftR(C* a)
{
    if (LR == 3) dft8<INV>(a); else if (LR == 2) dft4<INV>(a); else dft2<INV>(a);
}

template <typename C> __device__ __forceinline__ C ldg_c(const C* p) { return __ldg(p); }

// One pass over the tile.  LR = log2 radix, ls = log2 S (stride between butterfly legs, in points).
// tw: table exp(-2 pi i k / Ntab); lt = log2(Ntab / L)  (so w_L^j = tw[j << lt]).
template <typename T, int LR, bool INV>
__device__ __forceinline__ void fft_pass(typename cx_of<T>::type* s, int log2L, int ls, int B,
                                         const typename cx_of<T>::type* __restrict__ tw, int lt,
                                         int tid, int nthr)
{
    using C = typename cx_of<T>::type;
    constexpr int RB = cx_of<T>::ROWBITS;
    constexpr int R = 1 << LR;
    const int nb = (B << log2L) >> LR;           // butterflies in the tile
    const int S = 1 << ls;
    const int ltw = log2L - LR - ls + lt;        // w_n^j = tw[j << ltw],  n = R*S
    const bool pow2B = (B & (B - 1)) == 0;
    const int lB = 31 - __clz(B);
    for (int t = tid; t < nb; t += nthr) {
        int i, b;
        if (pow2B) { i = t >> lB; b = t & (B - 1); } else { i = t / B; b = t - i * B; }
        const int lo = i & (S - 1);
        const int p0 = ((i >> ls) << (ls + LR)) + lo;
        C a[R];
        int addr[R];
#pragma unroll
        for (int r = 0; r < R; ++r) { addr[r] = swz<RB>((p0 + (r << ls)) * B + b); a[r] = s[addr[r]]; }
        if (!INV) {
            dftR<LR, false>(a);
            if (ls > 0) {
                const int j = lo << ltw;
                if (LR == 3) {
                    const C w1 = ldg_c(tw + j), w2 = ldg_c(tw + 2 * j), w4 = ldg_c(tw + 4 * j);
                    const C w3 = cmul(w1, w2), w5 = cmul(w1, w4), w6 = cmul(w2, w4), w7 = cmul(w3, w4);
                    a[1] = cmul(a[1], w1); a[2] = cmul(a[2], w2); a[3] = cmul(a[3], w3); a[4] = cmul(a[4], w4);
                    a[5] = cmul(a[5], w5); a[6] = cmul(a[6], w6); a[7] = cmul(a[7], w7);
                } else if (LR == 2) {
                    const C w1 = ldg_c(tw + j), w2 = ldg_c(tw + 2 * j); const C w3 = cmul(w1, w2);
                    a[1] = cmul(a[1], w1); a[2] = cmul(a[2], w2); a[3] = cmul(a[3], w3);
                } else { a[1] = cmul(a[1], ldg_c(tw + j)); }
            }
        } else {
            if (ls > 0) {
                const int j = lo << ltw;
                if (LR == 3) {
                    const C w1 = ldg_c(tw + j), w2 = ldg_c(tw + 2 * j), w4 = ldg_c(tw + 4 * j);
                    const C w3 = cmul(w1, w2), w5 = cmul(w1, w4), w6 = cmul(w2, w4), w7 = cmul(w3, w4);
                    a[1] = cmulc(a[1], w1); a[2] = cmulc(a[2], w2); a[3] = cmulc(a[3], w3); a[4] = cmulc(a[4], w4);
                    a[5] = cmulc(a[5], w5); a[6] = cmulc(a[6], w6); a[7] = cmulc(a[7], w7);
                } else if (LR == 2) {
                    const C w1 = ldg_c(tw + j), w2 = ldg_c(tw + 2 * j); const C w3 = cmul(w1, w2);
                    a[1] = cmulc(a[1], w1); a[2] = cmulc(a[2], w2); a[3] = cmulc(a[3], w3);
                } else { a[1] = cmulc(a[1], ldg_c(tw + j)); }
            }
            dftR<LR, true>(a);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) s[addr[r]] = a[r];
    }
}

// All passes of a length-2^log2L transform on the tile s[L][B].  Caller has synchronised before
// (tile fully written); on return the tile is synchronised (all threads see the result).
template <typename T, bool INV>
__device__ __forceinline__ void fft_tile(typename cx_of<T>::type* s, int log2L, int B,
                                         const typename cx_of<T>::type* __restrict__ tw, int lt,
                                         int tid, int nthr)
{
    const int n8 = log2L / 3, rem = log2L % 3;
    if (!INV) {
        int ls = log2L;
        for (int i = 0; i < n8; ++i) { ls -= 3; fft_pass<T, 3, false>(s, log2L, ls, B, tw, lt, tid, nthr); __syncthreads(); }
        if (rem == 2) { fft_pass<T, 2, false>(s, log2L, 0, B, tw, lt, tid, nthr); __syncthreads(); }
        else if (rem == 1) { fft_pass<T, 1, false>(s, log2L, 0, B, tw, lt, tid, nthr); __syncthreads(); }
    } else {
        if (rem == 2) { fft_pass<T, 2, true>(s, log2L, 0, B, tw, lt, tid, nthr); __syncthreads(); }
        else if (rem == 1) { fft_pass<T, 1, true>(s, log2L, 0, B, tw, lt, tid, nthr); __syncthreads(); }
        int ls = rem;
        for (int i = 0; i < n8; ++i) { fft_pass<T, 3, true>(s, log2L, ls, B, tw, lt, tid, nthr); __syncthreads(); ls += 3; }
    }
}

}  // namespace demag
