// fft_core.cuh -- in-shared-memory batched power-of-two FFT used by every stage of the
// demagnetizing-field convolution ("N and M are first transformed using a FFT";
// Appendix A :296-321 xFFT / yFFT / zFFT).  sm_100a only; no cuFFT.
//
// A tile is a logical array  s[p][b]  of complex numbers, p = 0..L-1 the transform axis, b = 0..B-1
// the batch (independent lines), stored at  p*pitch + b.  Two addressing modes:
//   SWZ = false  batch-fastest tiles with >= 16 lines (or an odd pitch): a half warp touches 16
//                consecutive batch slots, so every access is conflict free with plain addressing;
//   SWZ = true   few long lines (B < 16): the flattened index is XOR-swizzled so that unit-stride and
//                power-of-two-strided accesses both spread over the banks (no padding bytes).
//
// Forward  = decimation in frequency, in place, natural order in  -> digit-reversed order out.
// Inverse  = decimation in time,      in place, digit-reversed in -> natural order out.
// The convolution never undoes the permutation in shared memory: loaders / storers address the tile
// through pos_of_freq().  Neither direction scales; 1/(Nx Ny Nz) lives in the kernel spectrum (R3).
//
// fp32 complex arithmetic uses Blackwell's packed f32x2 instructions (FADD2 / FMUL2 / FFMA2): one
// issue slot per complex add, two per complex multiply.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace demag {

extern __shared__ __align__(16) unsigned char demag_smem[];

template <typename T> struct cx_of;
template <> struct cx_of<float>  { using type = float2;  static constexpr int ROWBITS = 4; };
template <> struct cx_of<double> { using type = double2; static constexpr int ROWBITS = 3; };

template <typename C> __device__ __forceinline__ C cmake(decltype(C::x) a, decltype(C::x) b) { C r; r.x = a; r.y = b; return r; }

// ---- packed fp32 pair primitives ---------------------------------------------------------------
__device__ __forceinline__ float2 p_add(float2 a, float2 b)
{
    float2 r;
    asm("{.reg .b64 ra, rb, rc; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; add.rn.f32x2 rc, ra, rb; mov.b64 {%0,%1}, rc;}"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 p_sub(float2 a, float2 b)
{
    float2 r;
    asm("{.reg .b64 ra, rb, rc; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; sub.rn.f32x2 rc, ra, rb; mov.b64 {%0,%1}, rc;}"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 p_mul(float2 a, float2 b)
{
    float2 r;
    asm("{.reg .b64 ra, rb, rc; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; mul.rn.f32x2 rc, ra, rb; mov.b64 {%0,%1}, rc;}"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 p_fma(float2 a, float2 b, float2 c)
{
    float2 r;
    asm("{.reg .b64 ra, rb, rc, rd; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; mov.b64 rc, {%6,%7}; fma.rn.f32x2 rd, ra, rb, rc; mov.b64 {%0,%1}, rd;}"
        : "=f"(r.x), "=f"(r.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return r;
}
__device__ __forceinline__ double2 p_add(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 p_sub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 p_mul(double2 a, double2 b) { return make_double2(a.x * b.x, a.y * b.y); }
__device__ __forceinline__ double2 p_fma(double2 a, double2 b, double2 c) { return make_double2(fma(a.x, b.x, c.x), fma(a.y, b.y, c.y)); }

// ---- complex helpers -----------------------------------------------------------------------------
template <typename C> __device__ __forceinline__ C cadd(C a, C b) { return p_add(a, b); }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { return p_sub(a, b); }
template <typename C> __device__ __forceinline__ C cswap(C a) { return cmake<C>(a.y, a.x); }
// a * w
template <typename C> __device__ __forceinline__ C cmul(C a, C w)
{
    return p_fma(cmake<C>(a.x, a.x), w, p_mul(cmake<C>(a.y, a.y), cmake<C>(-w.y, w.x)));
}
// a * conj(w)
template <typename C> __device__ __forceinline__ C cmulc(C a, C w)
{
    return p_fma(cmake<C>(a.x, a.x), cmake<C>(w.x, -w.y), p_mul(cmake<C>(a.y, a.y), cmake<C>(w.y, w.x)));
}
// a + (-i) b  (forward rotation)  /  a + (+i) b
template <typename C> __device__ __forceinline__ C cadd_mi(C a, C b)
{
    using T = decltype(C::x);
    return p_fma(cswap(b), cmake<C>((T)1, (T)-1), a);
}
template <typename C> __device__ __forceinline__ C cadd_pi(C a, C b)
{
    using T = decltype(C::x);
    return p_fma(cswap(b), cmake<C>((T)-1, (T)1), a);
}
// a + rot(b), a - rot(b) with rot = multiplication by -i (forward) or +i (inverse)
template <bool INV, typename C> __device__ __forceinline__ C cadd_rot(C a, C b) { return INV ? cadd_pi(a, b) : cadd_mi(a, b); }
template <bool INV, typename C> __device__ __forceinline__ C csub_rot(C a, C b) { return INV ? cadd_mi(a, b) : cadd_pi(a, b); }

// XOR swizzle of the flattened element index: rows of 2^ROWBITS elements (= 128 bytes), the in-row
// index is XORed with the folded row number.
template <int ROWBITS> __device__ __forceinline__ int swz(int q)
{
    const int r = q >> ROWBITS;
    const int f = (r ^ (r >> ROWBITS) ^ (r >> (2 * ROWBITS)) ^ (r >> (3 * ROWBITS))) & ((1 << ROWBITS) - 1);
    return q ^ f;
}
template <bool SWZ, int ROWBITS> __device__ __forceinline__ int taddr(int q) { return SWZ ? swz<ROWBITS>(q) : q; }

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
// HALF_IN: the upper half of the inputs is known to be zero (zero padding).
template <bool INV, bool HALF_IN, typename C> __device__ __forceinline__ void dft2(C* a)
{
    if (HALF_IN) { a[1] = a[0]; return; }
    const C t = a[0]; a[0] = cadd(t, a[1]); a[1] = csub(t, a[1]);
}
template <bool INV, bool HALF_IN, typename C> __device__ __forceinline__ void dft4(C* a)
{
    C d0, d2;
    if (HALF_IN) { d0 = a[0]; d2 = a[0]; } else { d0 = cadd(a[0], a[2]); d2 = csub(a[0], a[2]); }
    C d1, t;
    if (HALF_IN) { d1 = a[1]; t = a[1]; } else { d1 = cadd(a[1], a[3]); t = csub(a[1], a[3]); }
    a[0] = cadd(d0, d1); a[2] = csub(d0, d1);
    a[1] = cadd_rot<INV>(d2, t); a[3] = csub_rot<INV>(d2, t);
}
template <bool INV, bool HALF_IN, typename C> __device__ __forceinline__ void dft8(C* a)
{
    using T = decltype(C::x);
    const T h = (T)0.70710678118654752440;
    C e[4], o[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        if (HALF_IN) { e[j] = a[j]; o[j] = a[j]; } else { e[j] = cadd(a[j], a[j + 4]); o[j] = csub(a[j], a[j + 4]); }
    }
    // o[1] *= w8, o[3] *= w8^3 (forward w8 = exp(-i pi/4)); o[2]'s rotation is folded into the dft4 below
    const C hh = cmake<C>(h, h);
    if (!INV) {
        o[1] = p_fma(cswap(o[1]), cmake<C>(h, -h), p_mul(o[1], hh));            // (x+y, y-x) h
        o[3] = p_fma(cswap(o[3]), cmake<C>(h, -h), p_mul(o[3], cmake<C>(-h, -h)));  // (y-x, -x-y) h
    } else {
        o[1] = p_fma(cswap(o[1]), cmake<C>(-h, h), p_mul(o[1], hh));            // (x-y, x+y) h
        o[3] = p_fma(cswap(o[3]), cmake<C>(-h, h), p_mul(o[3], cmake<C>(-h, -h)));  // (-x-y, x-y) h
    }
    dft4<INV, false>(e);
    {   // dft4 of (o0, o1, rot(o2), o3) with the rotation of o2 folded in
        const C d0 = cadd_rot<INV>(o[0], o[2]), d2 = csub_rot<INV>(o[0], o[2]);
        const C d1 = cadd(o[1], o[3]), t = csub(o[1], o[3]);
        o[0] = cadd(d0, d1); o[2] = csub(d0, d1);
        o[1] = cadd_rot<INV>(d2, t); o[3] = csub_rot<INV>(d2, t);
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) { a[2 * j] = e[j]; a[2 * j + 1] = o[j]; }
}
template <int LR, bool INV, bool HALF_IN, typename C> __device__ __forceinline__ void dftR(C* a)
{
    if (LR == 3) dft8<INV, HALF_IN>(a); else if (LR == 2) dft4<INV, HALF_IN>(a); else if (LR == 1) dft2<INV, HALF_IN>(a);
}

// a[m] *= w^m (forward) or conj(w)^m (inverse), m = 1..R-1, w^m read / derived from the table at j*m.
// UNI: the index j is the same for (nearly) all lanes of a warp (lines-fastest thread mapping), so every power is
// read directly (broadcast loads, one sector each); otherwise w, w^2, w^4 are read and the rest derived.
template <int LR, bool INV, bool UNI, typename C>
__device__ __forceinline__ void twiddle(C* a, const C* __restrict__ tw, int j)
{
    if (LR == 3) {
        C w1, w2, w3, w4, w5, w6, w7;
        if (UNI) {
            w1 = __ldg(tw + j); w2 = __ldg(tw + 2 * j); w3 = __ldg(tw + 3 * j); w4 = __ldg(tw + 4 * j);
            w5 = __ldg(tw + 5 * j); w6 = __ldg(tw + 6 * j); w7 = __ldg(tw + 7 * j);
        } else {
            w1 = __ldg(tw + j); w2 = __ldg(tw + 2 * j); w4 = __ldg(tw + 4 * j);
            w3 = cmul(w1, w2); w5 = cmul(w1, w4); w6 = cmul(w2, w4); w7 = cmul(w3, w4);
        }
        if (!INV) { a[1] = cmul(a[1], w1); a[2] = cmul(a[2], w2); a[3] = cmul(a[3], w3); a[4] = cmul(a[4], w4);
                    a[5] = cmul(a[5], w5); a[6] = cmul(a[6], w6); a[7] = cmul(a[7], w7); }
        else      { a[1] = cmulc(a[1], w1); a[2] = cmulc(a[2], w2); a[3] = cmulc(a[3], w3); a[4] = cmulc(a[4], w4);
                    a[5] = cmulc(a[5], w5); a[6] = cmulc(a[6], w6); a[7] = cmulc(a[7], w7); }
    } else if (LR == 2) {
        const C w1 = __ldg(tw + j), w2 = __ldg(tw + 2 * j); const C w3 = UNI ? __ldg(tw + 3 * j) : cmul(w1, w2);
        if (!INV) { a[1] = cmul(a[1], w1); a[2] = cmul(a[2], w2); a[3] = cmul(a[3], w3); }
        else      { a[1] = cmulc(a[1], w1); a[2] = cmulc(a[2], w2); a[3] = cmulc(a[3], w3); }
    } else if (LR == 1) {
        const C w1 = __ldg(tw + j);
        a[1] = INV ? cmulc(a[1], w1) : cmul(a[1], w1);
    }
}

// One in-place pass over the tile.  LR = log2 radix, ls = log2 S (stride between butterfly legs, in
// points).  tw: table exp(-2 pi i k / Ntab); lt = log2(Ntab / L)  (so w_L^j = tw[j << lt]).
template <typename T, int LR, bool INV, bool SWZ>
__device__ __forceinline__ void fft_pass(typename cx_of<T>::type* s, int log2L, int ls, int B, int pitch,
                                         const typename cx_of<T>::type* __restrict__ tw, int lt,
                                         int tid, int nthr)
{
    using C = typename cx_of<T>::type;
    constexpr int RB = cx_of<T>::ROWBITS;
    constexpr int R = 1 << LR;
    const int nb = (B << log2L) >> LR;           // butterflies in the tile
    const int S = 1 << ls;
    const int ltw = log2L - LR - ls + lt;        // w_n^j = tw[j << ltw],  n = R*S
    const int stride = pitch << ls;
    // lines fastest: butterfly t = i*B + b; (i, b) advance incrementally by nthr per iteration (no division in the loop)
    int b = tid % B, i = tid / B;
    const int db = nthr % B, di = nthr / B;
    for (int t = tid; t < nb; t += nthr, b += db, i += di) {
        if (b >= B) { b -= B; ++i; }
        const int lo = i & (S - 1);
        const int p0 = ((i >> ls) << (ls + LR)) + lo;
        const int q0 = p0 * pitch + b;
        C a[R];
#pragma unroll
        for (int r = 0; r < R; ++r) a[r] = s[taddr<SWZ, RB>(q0 + r * stride)];
        if (!INV) {
            dftR<LR, false, false>(a);
            if (ls > 0) twiddle<LR, false, !SWZ>(a, tw, lo << ltw);
        } else {
            if (ls > 0) twiddle<LR, true, !SWZ>(a, tw, lo << ltw);
            dftR<LR, true, false>(a);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) s[taddr<SWZ, RB>(q0 + r * stride)] = a[r];
    }
}

// All passes of a length-2^log2L transform on the tile s[L][B].  Caller has synchronised before
// (tile fully written); on return the tile is synchronised (all threads see the result).
template <typename T, bool INV, bool SWZ>
__device__ __forceinline__ void fft_tile(typename cx_of<T>::type* s, int log2L, int B, int pitch,
                                         const typename cx_of<T>::type* __restrict__ tw, int lt,
                                         int tid, int nthr)
{
    const int n8 = log2L / 3, rem = log2L % 3;
    if (!INV) {
        int ls = log2L;
        for (int i = 0; i < n8; ++i) { ls -= 3; fft_pass<T, 3, false, SWZ>(s, log2L, ls, B, pitch, tw, lt, tid, nthr); __syncthreads(); }
        if (rem == 2) { fft_pass<T, 2, false, SWZ>(s, log2L, 0, B, pitch, tw, lt, tid, nthr); __syncthreads(); }
        else if (rem == 1) { fft_pass<T, 1, false, SWZ>(s, log2L, 0, B, pitch, tw, lt, tid, nthr); __syncthreads(); }
    } else {
        if (rem == 2) { fft_pass<T, 2, true, SWZ>(s, log2L, 0, B, pitch, tw, lt, tid, nthr); __syncthreads(); }
        else if (rem == 1) { fft_pass<T, 1, true, SWZ>(s, log2L, 0, B, pitch, tw, lt, tid, nthr); __syncthreads(); }
        int ls = rem;
        for (int i = 0; i < n8; ++i) { fft_pass<T, 3, true, SWZ>(s, log2L, ls, B, pitch, tw, lt, tid, nthr); __syncthreads(); ls += 3; }
    }
}

}  // namespace demag
