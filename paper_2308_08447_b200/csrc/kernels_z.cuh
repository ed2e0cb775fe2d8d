// kernels_z.cuh -- compile-time specialised z stage (K3) for the common sizes: same algorithm and data
// layout as k_z_mul in kernels.cuh (first forward pass from global, fused middle stage, last inverse pass
// to global), but Nz, the tile width TY and the block size are template constants, so every shared-memory
// offset is an immediate and every loop is unrolled.  ("z FFTs, kernel
// multiplications and z IFFTs are done in the same routine".)
#pragma once
#include "kernels.cuh"

namespace demag {

// in-place radix-2^LR pass, stride 2^LS, on a tile s[2^LL][B] (lines fastest), NT threads, NT % B == 0
template <typename T, int LR, bool INV, int LL, int LS, int B, int NT>
__device__ __forceinline__ void fft_pass_c(typename cx_of<T>::type* s, const typename cx_of<T>::type* __restrict__ tw, int tid)
{
    using C = typename cx_of<T>::type;
    constexpr int R = 1 << LR, S = 1 << LS;
    constexpr int NBF = (1 << (LL - LR));          // butterflies per line
    constexpr int G = NT / B;                      // butterflies processed per step across the block
    constexpr int LTW = LL - LR - LS;
    const int b = tid % B, i0 = tid / B;
#pragma unroll 1
    for (int k = 0; k < (NBF + G - 1) / G; ++k) {
        const int i = i0 + k * G;
        if ((NBF % G) != 0 && i >= NBF) break;
        const int lo = i & (S - 1);
        const int p0 = ((i >> LS) << (LS + LR)) + lo;
        C* d = s + p0 * B + b;
        C a[R];
#pragma unroll
        for (int r = 0; r < R; ++r) a[r] = d[r * S * B];
        if (!INV) {
            dftR<LR, false, false>(a);
            if (LS > 0) twiddle<LR, false, true>(a, tw, lo << LTW);
        } else {
            if (LS > 0) twiddle<LR, true, true>(a, tw, lo << LTW);
            dftR<LR, true, false>(a);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) d[r * S * B] = a[r];
    }
}

template <typename T, int LL, int B, int NT, int K, bool INV> struct MidPasses {
    // forward: passes k = 1 .. n8-1 in increasing k; inverse: decreasing k.  K counts down from n8-1 to 1.
    static __device__ __forceinline__ void run(typename cx_of<T>::type* s, const typename cx_of<T>::type* __restrict__ tw, int tid)
    {
        constexpr int n8 = LL / 3, rem = LL % 3;
        constexpr int npass = n8 + (rem ? 1 : 0);
        constexpr int kk = INV ? K : (npass - 1 - K);          // pass index in schedule order
        if (K >= 1 && K <= npass - 2) {
            if (!INV) {
                fft_pass_c<T, 3, false, LL, LL - 3 * (kk + 1), B, NT>(s, tw, tid);
                __syncthreads();
                MidPasses<T, LL, B, NT, K - 1, INV>::run(s, tw, tid);
            } else {
                fft_pass_c<T, 3, true, LL, LL - 3 * (kk + 1), B, NT>(s, tw, tid);
                __syncthreads();
                MidPasses<T, LL, B, NT, K - 1, INV>::run(s, tw, tid);
            }
        }
    }
};
template <typename T, int LL, int B, int NT, bool INV> struct MidPasses<T, LL, B, NT, 0, INV> {
    static __device__ __forceinline__ void run(typename cx_of<T>::type*, const typename cx_of<T>::type* __restrict__, int) {}
};

template <typename T, int LNZ, int TY, int NT>
__global__ void __launch_bounds__(NT, (sizeof(T) == 4 && NT * 2 <= 1024 ? 2 : 1)) k_z_mul_c(Geo g, int kx0, int nkx,
                                                typename cx_of<T>::type* __restrict__ W2,
                                                const T* __restrict__ K, size_t kcs,
                                                const typename cx_of<T>::type* __restrict__ twz)
{
    using C = typename cx_of<T>::type;
    constexpr int NZ = 1 << LNZ, B = 3 * TY;
    constexpr int n8 = LNZ / 3, rem = LNZ % 3, npass = n8 + (rem ? 1 : 0);
    constexpr int LRF = rem ? rem : 3;
    constexpr int RF = 1 << LRF;
    constexpr int S0 = NZ / 8, G = NT / B;
    static_assert(NT % B == 0 && npass >= 2, "block must be a multiple of 3*TY; Nz >= 16");
    C* s = reinterpret_cast<C*>(demag_smem);
    const int tid = threadIdx.x;
    const int tilesY = g.Ny / TY;
    const int kyt = blockIdx.x % tilesY, kxl = blockIdx.x / tilesY;
    const int ky0 = kyt * TY;
    const int kx = kx0 + kxl;
    const size_t cstride = (size_t)nkx * g.nz * g.Ny;
    C* base = W2 + ((size_t)kxl * g.nz) * g.Ny + ky0;
    const int b = tid % B, i0 = tid / B;
    const int c = b / TY, ty = b - c * TY;
    C* gcol = base + c * cstride + ty;
    const bool padded = g.Nz != g.nz;
    const size_t Ny = g.Ny;
    // ---- first forward pass straight from global (zero padding: upper half never loaded)
#pragma unroll 1
    for (int k = 0; k < (S0 + G - 1) / G; ++k) {
        const int i = i0 + k * G;
        if ((S0 % G) != 0 && i >= S0) break;
        C a[8];
        if (padded) {
#pragma unroll
            for (int r = 0; r < 4; ++r) a[r] = gcol[(size_t)(i + r * S0) * Ny];
            dft8<false, true>(a);
        } else {
#pragma unroll
            for (int r = 0; r < 8; ++r) a[r] = gcol[(size_t)(i + r * S0) * Ny];
            dft8<false, false>(a);
        }
        twiddle<3, false, true>(a, twz, i);
        C* d = s + i * B + b;
#pragma unroll
        for (int r = 0; r < 8; ++r) d[r * S0 * B] = a[r];
    }
    __syncthreads();
    // forward middle passes: schedule index 1 .. npass-2  (K runs npass-2 .. 1 with kk = npass-1-K)
    MidPasses<T, LNZ, B, NT, (npass >= 3 ? npass - 2 : 0), false>::run(s, twz, tid);
    // ---- fused middle stage: last forward pass, multiply, first inverse pass; thread = (butterfly, ky), 3 comps
    {
        constexpr int GF = NT / TY, NBF = NZ / RF;
        const int tyf = tid % TY, if0 = tid / TY;
#pragma unroll 1
        for (int i = if0; i < NBF; i += GF) {
            const int p0 = i << LRF;
            C a[3][RF];
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) {
#pragma unroll
                for (int m = 0; m < RF; ++m) a[cc][m] = s[(p0 + m) * B + cc * TY + tyf];
                dftR<LRF, false, false>(a[cc]);
            }
            const int kb = freq_of_pos(p0, LNZ);
#pragma unroll
            for (int m = 0; m < RF; ++m) {
                const KernelVals<T> kv = load_kernel<T>(g, K, kcs, kx, ky0 + tyf, kb + m * (NZ >> LRF));
                apply_kernel(kv, a[0][m], a[1][m], a[2][m]);
            }
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) {
                dftR<LRF, true, false>(a[cc]);
#pragma unroll
                for (int m = 0; m < RF; ++m) s[(p0 + m) * B + cc * TY + tyf] = a[cc][m];
            }
        }
    }
    __syncthreads();
    MidPasses<T, LNZ, B, NT, (npass >= 3 ? npass - 2 : 0), true>::run(s, twz, tid);
    // ---- last inverse pass straight to global, keeping z < nz (the crop)
#pragma unroll 1
    for (int k = 0; k < (S0 + G - 1) / G; ++k) {
        const int i = i0 + k * G;
        if ((S0 % G) != 0 && i >= S0) break;
        C a[8];
        const C* d = s + i * B + b;
#pragma unroll
        for (int r = 0; r < 8; ++r) a[r] = d[r * S0 * B];
        twiddle<3, true, true>(a, twz, i);
        dft8<true, false>(a);
#pragma unroll
        for (int r = 0; r < 8; ++r) if (r < 4 || !padded) gcol[(size_t)(i + r * S0) * Ny] = a[r];
    }
}

}  // namespace demag
