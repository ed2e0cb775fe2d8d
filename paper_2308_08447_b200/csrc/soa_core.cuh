// soa_core.cuh -- "two lines per thread" complex arithmetic for the fast FFT-convolution kernels (kernels_v2.cuh).
//
// Every stage of the convolution (Appendix A :296-326) is a batch of independent 1D transforms
// ("lines").  A thread always works on the SAME element of TWO lines at once and keeps it as a quad
//     CQ = { re(line0), re(line1), im(line0), im(line1) }
// so that every complex operation is a pair of Blackwell packed-fp32 instructions (FADD2 / FMUL2 / FFMA2 act on
// the two lines), a multiplication by -i / +i is free (swap the roles of re and im, flip one sign inside the
// following add), a twiddle multiplication costs 4 packed instructions for 2 lines, and one 128-bit shared or
// global access moves one point of both lines.  In fp64 the same code runs with scalar pairs.
//
// DFT conventions: forward exp(-2 pi i nk/R), inverse exp(+2 pi i nk/R), unnormalised; natural order in and out.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#if defined(__CUDACC__)
#define DM_HD __host__ __device__ __forceinline__
#define DM_HDC __host__ __device__ constexpr
#else
#define DM_HD inline
#define DM_HDC constexpr
#endif

namespace demag {
namespace v2 {

template <typename T> struct vec2;
template <> struct vec2<float>  { using type = float2; };
template <> struct vec2<double> { using type = double2; };

// ---- pair primitives (packed on the device in fp32) ------------------------------------------------
DM_HD float2 vadd(float2 a, float2 b)
{
#ifdef __CUDA_ARCH__
    return __fadd2_rn(a, b);
#else
    return make_float2(a.x + b.x, a.y + b.y);
#endif
}
DM_HD float2 vneg(float2 a) { return make_float2(-a.x, -a.y); }
DM_HD float2 vsub(float2 a, float2 b)
{
#ifdef __CUDA_ARCH__
    return __fadd2_rn(a, vneg(b));
#else
    return make_float2(a.x - b.x, a.y - b.y);
#endif
}
DM_HD float2 vmul(float2 a, float2 b)
{
#ifdef __CUDA_ARCH__
    return __fmul2_rn(a, b);
#else
    return make_float2(a.x * b.x, a.y * b.y);
#endif
}
DM_HD float2 vfma(float2 a, float2 b, float2 c)
{
#ifdef __CUDA_ARCH__
    return __ffma2_rn(a, b, c);
#else
    return make_float2(a.x * b.x + c.x, a.y * b.y + c.y);
#endif
}
DM_HD double2 vadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
DM_HD double2 vneg(double2 a) { return make_double2(-a.x, -a.y); }
DM_HD double2 vsub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
DM_HD double2 vmul(double2 a, double2 b) { return make_double2(a.x * b.x, a.y * b.y); }
DM_HD double2 vfma(double2 a, double2 b, double2 c)
{
#ifdef __CUDA_ARCH__
    return make_double2(fma(a.x, b.x, c.x), fma(a.y, b.y, c.y));
#else
    return make_double2(a.x * b.x + c.x, a.y * b.y + c.y);
#endif
}
DM_HD float2 vdup(float a) { return make_float2(a, a); }
DM_HD double2 vdup(double a) { return make_double2(a, a); }

// ---- the quad: one complex point of two lines --------------------------------------------------------
template <typename T> struct alignas(4 * sizeof(T)) CQ {
    typename vec2<T>::type re, im;
};

template <typename T> DM_HD CQ<T> cq_zero()
{
    CQ<T> r; r.re = vdup((T)0); r.im = vdup((T)0); return r;
}
template <typename T> DM_HD CQ<T> cadd(CQ<T> a, CQ<T> b) { CQ<T> r; r.re = vadd(a.re, b.re); r.im = vadd(a.im, b.im); return r; }
template <typename T> DM_HD CQ<T> csub(CQ<T> a, CQ<T> b) { CQ<T> r; r.re = vsub(a.re, b.re); r.im = vsub(a.im, b.im); return r; }
// a + (-i) b   and   a + (+i) b
template <typename T> DM_HD CQ<T> cadd_mi(CQ<T> a, CQ<T> b) { CQ<T> r; r.re = vadd(a.re, b.im); r.im = vsub(a.im, b.re); return r; }
template <typename T> DM_HD CQ<T> cadd_pi(CQ<T> a, CQ<T> b) { CQ<T> r; r.re = vsub(a.re, b.im); r.im = vadd(a.im, b.re); return r; }
// a + rot(b), a - rot(b); rot = multiplication by -i (forward) or +i (inverse)
template <bool INV, typename T> DM_HD CQ<T> cadd_rot(CQ<T> a, CQ<T> b) { return INV ? cadd_pi(a, b) : cadd_mi(a, b); }
template <bool INV, typename T> DM_HD CQ<T> csub_rot(CQ<T> a, CQ<T> b) { return INV ? cadd_mi(a, b) : cadd_pi(a, b); }
// a * w  and  a * conj(w); w.re = (wr, wr), w.im = (wi, wi)
template <typename T> DM_HD CQ<T> cmul(CQ<T> a, CQ<T> w)
{
    CQ<T> r;
    r.re = vfma(a.re, w.re, vneg(vmul(a.im, w.im)));
    r.im = vfma(a.re, w.im, vmul(a.im, w.re));
    return r;
}
template <typename T> DM_HD CQ<T> cmulc(CQ<T> a, CQ<T> w)
{
    CQ<T> r;
    r.re = vfma(a.re, w.re, vmul(a.im, w.im));
    r.im = vfma(a.im, w.re, vneg(vmul(a.re, w.im)));
    return r;
}
template <bool INV, typename T> DM_HD CQ<T> ctw(CQ<T> a, CQ<T> w) { return INV ? cmulc(a, w) : cmul(a, w); }
// a * (wr + i wi) for compile-time-like scalar constants (forward); inverse uses the conjugate
template <bool INV, typename T> DM_HD CQ<T> cmul_const(CQ<T> a, T wr, T wi)
{
    CQ<T> w; w.re = vdup(wr); w.im = vdup(wi);
    return INV ? cmulc(a, w) : cmul(a, w);
}
// a * h(1 - i) (forward) / a * h(1 + i) (inverse), h = 1/sqrt 2:   3 pair operations
template <bool INV, typename T> DM_HD CQ<T> cmul_w8(CQ<T> a)
{
    const typename vec2<T>::type h = vdup((T)0.70710678118654752440);
    const typename vec2<T>::type t = vmul(a.re, h);
    CQ<T> r;
    if (!INV) { r.re = vfma(a.im, h, t); r.im = vfma(a.im, h, vneg(t)); }          // h(re+im), h(im-re)
    else      { r.re = vfma(vneg(a.im), h, t); r.im = vfma(a.im, h, t); }          // h(re-im), h(re+im)
    return r;
}
// a * h(-1 - i) (forward) / a * h(-1 + i) (inverse)
template <bool INV, typename T> DM_HD CQ<T> cmul_w8_3(CQ<T> a)
{
    const typename vec2<T>::type h = vdup((T)0.70710678118654752440);
    const typename vec2<T>::type t = vmul(a.re, h);
    CQ<T> r;
    if (!INV) { r.re = vfma(a.im, h, vneg(t)); r.im = vfma(vneg(a.im), h, vneg(t)); }   // h(im-re), -h(re+im)
    else      { r.re = vfma(vneg(a.im), h, vneg(t)); r.im = vfma(vneg(a.im), h, t); }   // -h(re+im), h(re-im)
    return r;
}

// ---- butterflies: natural order in -> natural order out, unnormalised ---------------------------------
// HALF_IN: the upper half of the inputs is zero (zero padding) and is never read.
template <bool INV, bool HALF_IN, typename T> DM_HD void dft2(CQ<T>* a)
{
    if (HALF_IN) { a[1] = a[0]; return; }
    const CQ<T> t = a[0]; a[0] = cadd(t, a[1]); a[1] = csub(t, a[1]);
}
template <bool INV, bool HALF_IN, typename T> DM_HD void dft4(CQ<T>* a)
{
    CQ<T> d0, d2, d1, t;
    if (HALF_IN) { d0 = a[0]; d2 = a[0]; d1 = a[1]; t = a[1]; }
    else { d0 = cadd(a[0], a[2]); d2 = csub(a[0], a[2]); d1 = cadd(a[1], a[3]); t = csub(a[1], a[3]); }
    a[0] = cadd(d0, d1); a[2] = csub(d0, d1);
    a[1] = cadd_rot<INV>(d2, t); a[3] = csub_rot<INV>(d2, t);
}
template <bool INV, bool HALF_IN, typename T> DM_HD void dft8(CQ<T>* a)
{
    CQ<T> e[4], o[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        if (HALF_IN) { e[j] = a[j]; o[j] = a[j]; } else { e[j] = cadd(a[j], a[j + 4]); o[j] = csub(a[j], a[j + 4]); }
    }
    o[1] = cmul_w8<INV>(o[1]);
    o[3] = cmul_w8_3<INV>(o[3]);
    dft4<INV, false>(e);
    {   // dft4 of (o0, o1, rot(o2), o3): the rotation of o2 is folded into the adds
        const CQ<T> d0 = cadd_rot<INV>(o[0], o[2]), d2 = csub_rot<INV>(o[0], o[2]);
        const CQ<T> d1 = cadd(o[1], o[3]), t = csub(o[1], o[3]);
        o[0] = cadd(d0, d1); o[2] = csub(d0, d1);
        o[1] = cadd_rot<INV>(d2, t); o[3] = csub_rot<INV>(d2, t);
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) { a[2 * j] = e[j]; a[2 * j + 1] = o[j]; }
}
// 16 = 4 x 4:  n = 4 n1 + n2,  k = k1 + 4 k2;  y[n2][k1] = DFT4_{n1} a[4 n1 + n2];  y *= W16^(n2 k1);
// X[k1 + 4 k2] = DFT4_{n2} y[n2][k1].
template <bool INV, bool HALF_IN, typename T> DM_HD void dft16(CQ<T>* a)
{
    const T c1 = (T)0.92387953251128675613, s1 = (T)0.38268343236508977173;
    CQ<T> y[4][4];   // [k1][n2]
#pragma unroll
    for (int n2 = 0; n2 < 4; ++n2) {
        CQ<T> t[4];
        t[0] = a[n2]; t[1] = a[n2 + 4];
        if (!HALF_IN) { t[2] = a[n2 + 8]; t[3] = a[n2 + 12]; }
        dft4<INV, HALF_IN>(t);
#pragma unroll
        for (int k1 = 0; k1 < 4; ++k1) y[k1][n2] = t[k1];
    }
    // W16^(n2 k1): exponents 1,2,3 | 2,4,6 | 3,6,9
    y[1][1] = cmul_const<INV>(y[1][1], c1, -s1);
    y[1][2] = cmul_w8<INV>(y[1][2]);
    y[1][3] = cmul_const<INV>(y[1][3], s1, -c1);
    y[2][1] = cmul_w8<INV>(y[2][1]);
    /* y[2][2] *= W^4 = -i (fwd) / +i (inv): folded below */
    y[2][3] = cmul_w8_3<INV>(y[2][3]);
    y[3][1] = cmul_const<INV>(y[3][1], s1, -c1);
    y[3][2] = cmul_w8_3<INV>(y[3][2]);
    y[3][3] = cmul_const<INV>(y[3][3], -c1, s1);
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) {
        CQ<T> t[4] = {y[k1][0], y[k1][1], y[k1][2], y[k1][3]};
        if (k1 == 2) {   // dft4 of (t0, t1, rot(t2), t3)
            const CQ<T> d0 = cadd_rot<INV>(t[0], t[2]), d2 = csub_rot<INV>(t[0], t[2]);
            const CQ<T> d1 = cadd(t[1], t[3]), u = csub(t[1], t[3]);
            t[0] = cadd(d0, d1); t[2] = csub(d0, d1);
            t[1] = cadd_rot<INV>(d2, u); t[3] = csub_rot<INV>(d2, u);
        } else {
            dft4<INV, false>(t);
        }
#pragma unroll
        for (int k2 = 0; k2 < 4; ++k2) a[k1 + 4 * k2] = t[k2];
    }
}
// a * (-i) (forward) / a * (+i) (inverse)
template <bool INV, typename T> DM_HD CQ<T> crot(CQ<T> a)
{
    CQ<T> r;
    if (!INV) { r.re = a.im; r.im = vneg(a.re); } else { r.re = vneg(a.im); r.im = a.re; }
    return r;
}
// 32 = 2 x 16 (decimation in frequency): e[j] = a[j] + a[j+16], o[j] = (a[j] - a[j+16]) W32^j;
// X[2k] = DFT16(e)[k], X[2k+1] = DFT16(o)[k].  Used as the stride-1 (twiddle-free) pass of long y lines, where it
// removes one shared-memory sweep (512 = 16 . 32 instead of 8 . 8 . 8).
template <bool INV, bool HALF_IN, typename T> DM_HD void dft32(CQ<T>* a)
{
    const T c1 = (T)0.98078528040323044913, s1 = (T)0.19509032201612826785;
    const T c2 = (T)0.92387953251128675613, s2 = (T)0.38268343236508977173;
    const T c3 = (T)0.83146961230254523708, s3 = (T)0.55557023301960222474;
    CQ<T> o[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        if (HALF_IN) o[j] = a[j];
        else { const CQ<T> t = a[j]; a[j] = cadd(t, a[j + 16]); o[j] = csub(t, a[j + 16]); }
    }
    o[1] = cmul_const<INV>(o[1], c1, -s1);   o[2] = cmul_const<INV>(o[2], c2, -s2);   o[3] = cmul_const<INV>(o[3], c3, -s3);
    o[4] = cmul_w8<INV>(o[4]);
    o[5] = cmul_const<INV>(o[5], s3, -c3);   o[6] = cmul_const<INV>(o[6], s2, -c2);   o[7] = cmul_const<INV>(o[7], s1, -c1);
    o[8] = crot<INV>(o[8]);
    o[9] = cmul_const<INV>(o[9], -s1, -c1);  o[10] = cmul_const<INV>(o[10], -s2, -c2); o[11] = cmul_const<INV>(o[11], -s3, -c3);
    o[12] = cmul_w8_3<INV>(o[12]);
    o[13] = cmul_const<INV>(o[13], -c3, -s3); o[14] = cmul_const<INV>(o[14], -c2, -s2); o[15] = cmul_const<INV>(o[15], -c1, -s1);
    dft16<INV, false>(a);          // e, in place in a[0..15]
    dft16<INV, false>(o);
#pragma unroll
    for (int k = 15; k >= 0; --k) { a[2 * k + 1] = o[k]; a[2 * k] = a[k]; }
}
template <int LR, bool INV, bool HALF_IN, typename T> DM_HD void dftR(CQ<T>* a)
{
    if (LR == 5) dft32<INV, HALF_IN>(a);
    else if (LR == 4) dft16<INV, HALF_IN>(a);
    else if (LR == 3) dft8<INV, HALF_IN>(a);
    else if (LR == 2) dft4<INV, HALF_IN>(a);
    else if (LR == 1) dft2<INV, HALF_IN>(a);
}

// ---- radix schedule of a length-2^LL transform (shared by host table builders and kernels) -----------
// Decimation in frequency, in place: pass j has radix 2^lr(j) and stride S_j = L / (R_0 ... R_j); the inverse
// runs the same passes backwards (decimation in time).  POL selects the radix mix:
//   POL 0: radix 8 passes, remainder (2 or 4) LAST            (8,8,..,r)
//   POL 1: one leading radix-16 pass when LL % 3 == 1, leading radix 4 when LL % 3 == 2
//   POL 2: as many radix-16 as the remainder allows: LL%3==1 -> 16,8,..; LL%3==2 -> 16,16,8,.. (LL >= 8)
//   POL 3: radix 8 passes, remainder, radix 4 LAST (LL >= 4)
//   POL 5: radix 16 passes, remainder LAST
//   POL 7: two passes, radix 2^(LL-3) then radix 8 (LL = 7, 8)
//   POL 6: radix 16 passes, remainder, and a radix-32 LAST pass (LL >= 8; the y stage: the last forward / first
//          inverse pass runs straight against global memory, so 512 = 16 . 32 sweeps the tile once each way)
struct Sched {
    int n;          // number of passes
    int lr[6];      // log2 radix of each pass
    int ls[6];      // log2 stride of each pass
};
DM_HDC Sched make_sched(int LL, int POL)
{
    Sched s = {0, {0, 0, 0, 0, 0, 0}, {0, 0, 0, 0, 0, 0}};
    int rem = LL;
    if (POL == 0) {
        while (rem >= 3) { s.lr[s.n++] = 3; rem -= 3; }
        if (rem) s.lr[s.n++] = rem;
    } else if (POL == 5) {          // radix 16 passes, remainder LAST (long x rows: fewest sweeps)
        while (rem >= 4) { s.lr[s.n++] = 4; rem -= 4; }
        if (rem) s.lr[s.n++] = rem;
    } else if (POL == 7) {          // two passes: radix 2^(LL-3), then radix 8 (the even / odd half transforms of k_z_eo_v)
        s.lr[s.n++] = LL - 3; s.lr[s.n++] = 3;
    } else if (POL == 6) {          // radix 16 passes, remainder, and a radix-32 LAST pass
        rem -= 5;
        while (rem >= 4) { s.lr[s.n++] = 4; rem -= 4; }
        if (rem > 0) s.lr[s.n++] = rem;
        s.lr[s.n++] = 5;
    } else if (POL == 3) {          // radix 8 passes, remainder, and a radix-4 LAST pass (small fused z stage)
        rem -= 2;
        while (rem >= 3) { s.lr[s.n++] = 3; rem -= 3; }
        if (rem > 0) s.lr[s.n++] = rem;
        s.lr[s.n++] = 2;
    } else {
        const int b = LL % 3;
        if (POL == 2 && b == 2 && LL >= 8) { s.lr[s.n++] = 4; s.lr[s.n++] = 4; rem -= 8; }
        else if (b == 1 && LL >= 4) { s.lr[s.n++] = 4; rem -= 4; }
        else if (b != 0) { s.lr[s.n++] = b; rem -= b; }
        while (rem >= 3) { s.lr[s.n++] = 3; rem -= 3; }
    }
    int ls = LL;
    for (int j = 0; j < s.n; ++j) { ls -= s.lr[j]; s.ls[j] = ls; }
    return s;
}
// frequency held at position p after all forward passes (in-place DIF): pos = sum d_j S_j, freq = sum d_j W_j,
// W_j = R_0 ... R_{j-1}
DM_HDC int sched_freq_of_pos(const Sched& s, int p)
{
    int k = 0, w = 0;
    for (int j = 0; j < s.n; ++j) {
        const int d = (p >> s.ls[j]) & ((1 << s.lr[j]) - 1);
        k += d << w;
        w += s.lr[j];
    }
    return k;
}
DM_HDC int sched_pos_of_freq(const Sched& s, int k)
{
    int p = 0, w = 0;
    for (int j = 0; j < s.n; ++j) {
        const int d = (k >> w) & ((1 << s.lr[j]) - 1);
        p += d << s.ls[j];
        w += s.lr[j];
    }
    return p;
}

}  // namespace v2
}  // namespace demag
