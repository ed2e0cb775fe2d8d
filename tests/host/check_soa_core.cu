// Host-side check of the arithmetic building blocks of the fast kernel family (soa_core.cuh), compiled by
// tests/test_host_logic.py with nvcc and run on the CPU: every butterfly (radix 2/4/8/16/32, forward / inverse, full and
// zero-padded "half" input) against the DFT definition X[k] = sum_n x[n] exp(-+ 2 pi i n k / R), on both lines of the
// quads; every radix schedule is a bijection between positions and frequencies.  Prints "OK" or the first failure.
#include <cmath>
#include <complex>
#include <cstdio>
#include <vector>
#include "../../paper_2308_08447_b200/csrc/soa_core.cuh"
using namespace demag::v2;

template <int LR, bool INV, bool HALF> double butterfly_error()
{
    const int R = 1 << LR;
    CQ<double> a[32];
    std::complex<double> x0[32], x1[32];
    for (int i = 0; i < R; ++i) {
        const bool z = HALF && i >= R / 2;
        x0[i] = z ? 0 : std::complex<double>(sin(i * 1.3 + 0.2), cos(i * 0.7 + 1));
        x1[i] = z ? 0 : std::complex<double>(cos(i * 2.1 + 0.5), sin(i * 0.3 - 1));
        a[i].re = make_double2(x0[i].real(), x1[i].real());
        a[i].im = make_double2(x0[i].imag(), x1[i].imag());
    }
    if (HALF) for (int i = R / 2; i < R; ++i) { a[i].re = make_double2(1e30, 1e30); a[i].im = a[i].re; }   // must not be read
    dftR<LR, INV, HALF>(a);
    double err = 0;
    for (int k = 0; k < R; ++k) {
        std::complex<double> s0 = 0, s1 = 0;
        for (int n = 0; n < R; ++n) {
            const double ang = (INV ? 2 : -2) * M_PI * n * k / R;
            const std::complex<double> w(cos(ang), sin(ang));
            s0 += x0[n] * w; s1 += x1[n] * w;
        }
        err = fmax(err, std::abs(s0 - std::complex<double>(a[k].re.x, a[k].im.x)));
        err = fmax(err, std::abs(s1 - std::complex<double>(a[k].re.y, a[k].im.y)));
    }
    return err;
}
template <int LR> int check_radix()
{
    const double e[4] = {butterfly_error<LR, false, false>(), butterfly_error<LR, true, false>(),
                         butterfly_error<LR, false, true>(), butterfly_error<LR, true, true>()};
    for (int i = 0; i < 4; ++i)
        if (!(e[i] < (LR >= 5 ? 4e-13 : 1e-13))) {     // rounding: the sums reach ~2 R in magnitude
 printf("FAIL radix %d variant %d error %g\n", 1 << LR, i, e[i]); return 1; }
    return 0;
}
int main()
{
    int bad = check_radix<1>() + check_radix<2>() + check_radix<3>() + check_radix<4>() + check_radix<5>();
    // twiddle multiplication helpers
    {
        CQ<double> a, w;
        a.re = make_double2(0.3, -1.2); a.im = make_double2(0.7, 0.4);
        w.re = make_double2(0.6, 0.6); w.im = make_double2(-0.8, -0.8);
        const CQ<double> f = cmul(a, w), c = cmulc(a, w);
        const std::complex<double> A0(0.3, 0.7), A1(-1.2, 0.4), W(0.6, -0.8);
        if (std::abs(A0 * W - std::complex<double>(f.re.x, f.im.x)) > 1e-15 || std::abs(A1 * W - std::complex<double>(f.re.y, f.im.y)) > 1e-15 ||
            std::abs(A0 * std::conj(W) - std::complex<double>(c.re.x, c.im.x)) > 1e-15) { printf("FAIL cmul\n"); ++bad; }
    }
    for (int LL = 1; LL <= 13; ++LL)
        for (int pol : {0, 1, 2, 3, 5, 6}) {
            if (pol == 3 && LL < 4) continue;
            if (pol == 6 && LL < 8) continue;
            const Sched s = make_sched(LL, pol);
            int tot = 0;
            for (int j = 0; j < s.n; ++j) tot += s.lr[j];
            bool ok = tot == LL && s.n >= 1 && s.n <= 6 && s.ls[s.n - 1] == 0;
            std::vector<int> seen(1 << LL, 0);
            for (int p = 0; p < (1 << LL) && ok; ++p) {
                const int k = sched_freq_of_pos(s, p);
                ok = k >= 0 && k < (1 << LL) && sched_pos_of_freq(s, k) == p && seen[k]++ == 0;
            }
            if (!ok) { printf("FAIL schedule LL=%d policy=%d\n", LL, pol); ++bad; }
        }
    if (!bad) printf("OK\n");
    return bad ? 1 : 0;
}
