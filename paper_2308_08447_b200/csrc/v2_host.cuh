// v2_host.cuh -- host side of the fast path (kernels_v2.cuh): per-size launch configurations, twiddle tables,
// the plan-time pack of the kernel spectrum into the pair layout, and the launchers demag_apply calls.
#pragma once
#include <math.h>
#include <stdlib.h>
#include <vector>
#include "kernels_v2.cuh"

namespace demag {
namespace v2 {

// ---- launch configurations (compile-time, by log2 transform length) ---------------------------------------
// x stage (K1v / K5v): radix policy, row pairs per tile, threads
template <int LLC> struct XCfg { static constexpr int POL = 1, RP = 8, NT = 64; };
template <> struct XCfg<8>  { static constexpr int POL = 2, RP = 8, NT = 128; };
template <> struct XCfg<9>  { static constexpr int POL = 1, RP = 8, NT = 256; };
template <> struct XCfg<10> { static constexpr int POL = 1, RP = 4, NT = 256; };
template <> struct XCfg<11> { static constexpr int POL = 1, RP = 2, NT = 256; };
template <> struct XCfg<12> { static constexpr int POL = 5, RP = 1, NT = 256; };   // 16 . 16 . 16
template <> struct XCfg<13> { static constexpr int POL = 6, RP = 1, NT = 256; };   // 16 . 16 . 32 (nx = 8192: the paper's 7680-cell rows)
// y stage (K2v / K4v): radix policy, line pairs per tile, threads
template <int LNY> struct YCfg { static constexpr int POL = 1, BP = 8, NT = 64; };
template <> struct YCfg<8>  { static constexpr int POL = 1, BP = 8, NT = 128; };
template <> struct YCfg<9>  { static constexpr int POL = 1, BP = 8, NT = 256; };
template <> struct YCfg<10> { static constexpr int POL = 1, BP = 4, NT = 256; };
template <> struct YCfg<11> { static constexpr int POL = 1, BP = 2, NT = 256; };
template <> struct YCfg<12> { static constexpr int POL = 1, BP = 1, NT = 256; };
template <> struct YCfg<13> { static constexpr int POL = 1, BP = 1, NT = 512; };
// fp32 lines whose LAST pass -- the one that runs straight against global memory -- is radix 32 (policy 6): the tile is
// swept once each way instead of twice (512 = 16 . 32) or twice instead of three times (8192 = 16 . 16 . 32).  The
// radix-32 butterfly holds 32 quads (128 registers), so blocks are smaller.
template <int LNY> struct YCfg32 { static constexpr bool has = false; static constexpr int POL = 1, BP = 8, NT = 64; };
template <> struct YCfg32<9>  { static constexpr bool has = true; static constexpr int POL = 6, BP = 8, NT = 128; };   // 16 . 32
template <> struct YCfg32<13> { static constexpr bool has = true; static constexpr int POL = 6, BP = 1, NT = 256; };   // 16 . 16 . 32
// z stage (K3v): radix policy (the LAST pass is the fused one), ky columns per tile, threads, min blocks per SM
template <int LNZ> struct ZCfg { static constexpr int POL = 1, TY = 16, NT = 64, MINB = 1; };
template <> struct ZCfg<4>  { static constexpr int POL = 0, TY = 32, NT = 128, MINB = 1; };   // 8 . 2
template <> struct ZCfg<5>  { static constexpr int POL = 1, TY = 16, NT = 64,  MINB = 1; };   // 4 . 8
template <> struct ZCfg<6>  { static constexpr int POL = 1, TY = 16, NT = 128, MINB = 1; };   // 8 . 8
template <> struct ZCfg<7>  { static constexpr int POL = 1, TY = 8,  NT = 64,  MINB = 1; };   // 16 . 8
template <> struct ZCfg<8>  { static constexpr int POL = 1, TY = 4,  NT = 64,  MINB = 1; };   // 4 . 8 . 8
template <> struct ZCfg<9>  { static constexpr int POL = 1, TY = 4,  NT = 128, MINB = 1; };   // 8 . 8 . 8
template <> struct ZCfg<10> { static constexpr int POL = 1, TY = 2,  NT = 128, MINB = 1; };   // 16 . 8 . 8
template <> struct ZCfg<11> { static constexpr int POL = 1, TY = 1,  NT = 64,  MINB = 1; };   // 4 . 8 . 8 . 8
// fp64 (opt-in, DEMAG_PATH=fast): a quad is 32 bytes, so the same tile shapes would take twice the shared memory and halve
// the resident blocks; tiles of half the width keep the occupancy of the fp32 shapes (C3 fp64: 1.24 -> 1.02 ms; quarter
// width measured slower for every stage; the generic family, 1.06 ms, stays the default for fp64 plans)
template <int LLC> struct XCfgD { static constexpr int POL = XCfg<LLC>::POL, RP = (LLC >= 8 && XCfg<LLC>::RP >= 2) ? XCfg<LLC>::RP / 2 : XCfg<LLC>::RP, NT = XCfg<LLC>::NT; };
template <int LNY> struct YCfgD { static constexpr int POL = YCfg<LNY>::POL, BP = (LNY >= 9 && YCfg<LNY>::BP >= 2) ? YCfg<LNY>::BP / 2 : YCfg<LNY>::BP, NT = YCfg<LNY>::NT; };
template <int LNZ> struct ZCfgD { static constexpr int POL = ZCfg<LNZ>::POL, TY = (LNZ >= 6 && ZCfg<LNZ>::TY >= 2) ? ZCfg<LNZ>::TY / 2 : ZCfg<LNZ>::TY, NT = ZCfg<LNZ>::NT, MINB = ZCfg<LNZ>::MINB; };
template <typename F, typename D, typename T> struct CfgSel { using type = F; };
template <typename F, typename D> struct CfgSel<F, D, double> { using type = D; };

// quads of the y tile (skewed when the schedule has >= 2 passes, kernels_v2.cuh "tile addressing")
constexpr int y_tile_quads(int LNY, int POL, int BP)
{
    return tile_quads(tile_pe(BP | 1, make_sched(LNY, POL).n >= 2 ? 1 : 0, POL == 6), 1 << LNY, BP);
}
constexpr int x_tile_quads(int LLC, int POL, int RP) { return tile_quads(tile_pe(RP | 1, (RP < 8 && skew_ok(LLC, POL)) ? RP : 0, true), 1 << LLC, RP); }
constexpr int z_tile_quads(int LNZ, int POL, int TY) { return tile_quads(tile_pe(3 * TY, (TY <= 2 && skew_ok(LNZ, POL)) ? TY : 0), 1 << LNZ, 3 * TY); }
// W2v position p' of a y line -> in-place (digit-reversed) tile position: with >= 2 passes the last pass scatters
// output r of butterfly i to r * (Ny / R) + i
inline int y_w2_pos_to_tile_pos(int LNY, int POL, int pw)
{
    const Sched sc = make_sched(LNY, POL);
    if (sc.n < 2) return pw;
    const int lr = sc.lr[sc.n - 1], lnb = LNY - lr;
    return ((pw & ((1 << lnb) - 1)) << lr) + (pw >> lnb);
}
constexpr int kXMin = 4, kXMax = 13, kYMin = 4, kYMax = 13, kZMin = 2, kZMax = 11;

inline int x_rp_f(int lLc)
{
    switch (lLc) { case 10: return XCfg<10>::RP; case 11: return XCfg<11>::RP; case 12: return XCfg<12>::RP; case 13: return XCfg<13>::RP; default: return 8; }
}
inline int x_pol(int lLc) { return lLc == 8 ? XCfg<8>::POL : lLc == 12 ? XCfg<12>::POL : lLc == 13 ? XCfg<13>::POL : 1; }
inline bool y_has32(int lNy) { return lNy == 9 || lNy == 13; }
inline int y_pol(int lNy, bool y32 = false) { return y32 && y_has32(lNy) ? 6 : 1; }
inline int z_pol(int lNz) { return lNz == 4 ? ZCfg<4>::POL : 1; }
inline int x_rp(int lLc, size_t esz = 4) { const int r = x_rp_f(lLc); return (esz == 8 && lLc >= 8 && r >= 2) ? r / 2 : r; }
inline int z_ty_f(int lNz)
{
    switch (lNz) {
    case 0: case 2: case 3: return 1;
    case 4: return ZCfg<4>::TY; case 5: return ZCfg<5>::TY; case 6: return ZCfg<6>::TY; case 7: return ZCfg<7>::TY;
    case 8: return ZCfg<8>::TY; case 9: return ZCfg<9>::TY; case 10: return ZCfg<10>::TY; case 11: return ZCfg<11>::TY;
    default: return 1 << 30;
    }
}
inline int z_ty(int lNz, size_t esz = 4) { const int t = z_ty_f(lNz); return (esz == 8 && lNz >= 6 && t >= 2 && t < (1 << 30)) ? t / 2 : t; }

// Can the fast path run this geometry?  (all axes zero padded, sizes inside the instantiated range, tiles divide)
inline bool supported(int nx, int ny, int nz, int Nx, int Ny, int Nz, int lLc, int lNy, int lNz, size_t esz, int max_smem)
{
    const bool film = nz == 1 && Nz == 1;          // a one-cell-thick mesh has no z transform (R6): multiply only
    if (Nx != 2 * nx || Ny != 2 * ny || (Nz != 2 * nz && !film)) return false;
    if (lLc < kXMin || lLc > kXMax || lNy < kYMin || lNy > kYMax || ((lNz < kZMin || lNz > kZMax) && !film)) return false;
    if (ny % (2 * x_rp(lLc, esz)) != 0) return false;
    if (lNz >= 4 && Ny % z_ty(lNz, esz) != 0) return false;
    if (lNz < 4 && Ny < 32) return false;
    // shared memory of the y tile (the largest): Ny * (BP|1) quads
    int bp = lNy <= 9 ? 8 : lNy == 10 ? 4 : lNy == 11 ? 2 : 1;
    if (esz == 8 && lNy >= 9 && bp >= 2) bp /= 2;
    if ((size_t)y_tile_quads(lNy, y_pol(lNy), bp) * 4 * esz > (size_t)max_smem) return false;
    if ((size_t)x_tile_quads(lLc, x_pol(lLc), x_rp(lLc, esz)) * 4 * esz > (size_t)max_smem) return false;
    if (lNz >= 4 && (size_t)z_tile_quads(lNz, z_pol(lNz), z_ty(lNz, esz)) * 4 * esz > (size_t)max_smem) return false;
    return true;
}

// ---- twiddle tables ------------------------------------------------------------------------------------
// pass j of schedule (LL, POL): entries [(m-1) S + lo] = exp(-2 pi i lo m / (R S)), m = 1..R-1, lo = 0..S-1, stored as
// quads {wr, wr, wi, wi}.  All passes of one axis live in one device buffer.
template <typename T>
struct AxisTables {
    void* dev = nullptr;
    size_t bytes = 0;
    TwSet<T> set;
};
template <typename T>
cudaError_t build_axis_tables(int LL, int POL, int extra_post_Lc, AxisTables<T>* out, const CQ<T>** post,
                              int eo_N = 0, const CQ<T>** eo = nullptr)
{
    const Sched sc = make_sched(LL, POL);
    std::vector<T> h;
    size_t off[6] = {0, 0, 0, 0, 0, 0};
    bool has[6] = {false, false, false, false, false, false};
    const long double tp = 6.283185307179586476925286766559005768L;
    for (int j = 0; j < sc.n; ++j) {
        const int R = 1 << sc.lr[j], S = 1 << sc.ls[j];
        if (S == 1) continue;
        has[j] = true; off[j] = h.size();
        for (int m = 1; m < R; ++m)
            for (int lo = 0; lo < S; ++lo) {
                const long double a = tp * (long double)lo * (long double)m / ((long double)R * (long double)S);
                const T wr = (T)cosl(a), wi = (T)(-sinl(a));
                h.push_back(wr); h.push_back(wr); h.push_back(wi); h.push_back(wi);
            }
    }
    size_t post_off = h.size();
    if (extra_post_Lc > 0) {     // w^k = exp(-2 pi i k / (2 Lc)), k = 0..Lc/2 (the real-transform split)
        for (int k = 0; k <= extra_post_Lc / 2; ++k) {
            const long double a = tp * (long double)k / (2.0L * (long double)extra_post_Lc);
            T wr = (T)cosl(a), wi = (T)(-sinl(a));
            if (2 * k == extra_post_Lc) { wr = 0; wi = -1; }
            h.push_back(wr); h.push_back(wr); h.push_back(wi); h.push_back(wi);
        }
    }
    size_t eo_off = h.size();
    if (eo_N > 0) {              // w_N^z = exp(-2 pi i z / N), z = 0..N/2-1 (the odd half transform of k_z_eo_v)
        for (int z = 0; z < eo_N / 2; ++z) {
            const long double a = tp * (long double)z / (long double)eo_N;
            T wr = (T)cosl(a), wi = (T)(-sinl(a));
            if (4 * z == eo_N) { wr = 0; wi = -1; }
            h.push_back(wr); h.push_back(wr); h.push_back(wi); h.push_back(wi);
        }
    }
    if (h.empty()) h.resize(4, (T)0);
    out->bytes = h.size() * sizeof(T);
    cudaError_t e = cudaMalloc(&out->dev, out->bytes);
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(out->dev, h.data(), out->bytes, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
    for (int j = 0; j < 6; ++j) out->set.p[j] = has[j] ? reinterpret_cast<const CQ<T>*>((const T*)out->dev + off[j]) : nullptr;
    if (post) *post = extra_post_Lc > 0 ? reinterpret_cast<const CQ<T>*>((const T*)out->dev + post_off) : nullptr;
    if (eo) *eo = eo_N > 0 ? reinterpret_cast<const CQ<T>*>((const T*)out->dev + eo_off) : nullptr;
    return cudaSuccess;
}

inline int z_kt(int lNz, size_t esz = 4) { return lNz >= 4 ? z_ty(lNz, esz) : 32; }     // slot tile = the z kernel's column tile (32: register kernels)
// ---- plan-time pack of the transformed tensor into the pair layout -----------------------------------------
// A = real 3D transform of one component, [kz'][ky'][kx] (kx = 0..Lc).  Kv[q][slot / KT][kz'][chunk][slot % KT], lines (q, Lc-q)
// (kernels_v2.cuh "Kv").  ypos2freq[py] = y frequency stored at W2v position py (the y schedule's digit reversal);
// only the positions with ky <= Ny/2 are stored, at yslot[py] (the mirrored ones read the same slot with the sign of
// the y-odd components flipped in the kernel).
template <typename T>
__global__ void k_pack_kernel_v(const double* __restrict__ A, T* __restrict__ Kv, int comp, int Lc, int hq, int kpy, int kpz,
                                int Ny, int KT, int kst, const int* __restrict__ ypos2freq, const int* __restrict__ yslot, double scale, int q0)
{
    // hq pairs starting at pair q0 (several GPUs: K^(g) holds only its own kx range; else q0 = 0)
    const size_t n = (size_t)hq * kpz * Ny;
    const int hx = Lc + 1;
    constexpr int U = 16 / (int)sizeof(T), NCH = 12 / U;          // values per 16-byte chunk, chunks per entry
    const int j = sizeof(T) == 4 ? comp / 2 : comp, off = sizeof(T) == 4 ? (comp % 2) * 2 : 0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int py = (int)(i % Ny), kz = (int)((i / Ny) % kpz), q = (int)(i / ((size_t)Ny * kpz));
        const int ky = ypos2freq[py];
        if (2 * ky > Ny) continue;                                 // mirrored: shares the slot of Ny - ky
        const double* row = A + ((size_t)kz * kpy + ky) * hx;
        const int slot = yslot[py];
        T* d = Kv + ((((((size_t)q * kst + slot / KT) * kpz + kz) * NCH + j) * KT) + slot % KT) * U + off;
        d[0] = (T)(scale * row[q0 + q]);
        d[1] = (T)(scale * row[Lc - q0 - q]);
    }
}

// One-cell-thick meshes (k_z_v FILM): A = [ky'][kx] (kpz = 1).  Kf[q][ky'][chunk], y packed by symmetry (the kernel
// applies the mirror sign itself), components stored in the slots of the (x, z, y) line order:
// xx->xx, yy->zz, zz->yy, xy->xz, xz->xy, yz->yz.
template <typename T>
__global__ void k_pack_film_v(const double* __restrict__ A, T* __restrict__ Kf, int comp, int Lc, int hq, int kpy, double scale)
{
    const size_t n = (size_t)hq * kpy;
    const int hx = Lc + 1;
    constexpr int U = 16 / (int)sizeof(T), NCH = 12 / U;
    const int slot = comp == 1 ? 2 : comp == 2 ? 1 : comp == 3 ? 4 : comp == 4 ? 3 : comp;
    const int j = sizeof(T) == 4 ? slot / 2 : slot, off = sizeof(T) == 4 ? (slot % 2) * 2 : 0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int ky = (int)(i % kpy), q = (int)(i / kpy);
        const double* row = A + (size_t)ky * hx;
        T* d = Kf + (i * NCH + j) * U + off;
        d[0] = (T)(scale * row[q]);
        d[1] = (T)(scale * row[Lc - q]);
    }
}
inline int film_pol(int lNy) { return lNy == 4 ? 0 : (lNy == 8 || lNy == 11) ? 2 : 1; }   // 2048 = 16 . 16 . 8
inline bool film_supported(int nz, int Nz, int lNy, size_t esz, int max_smem)
{
    return nz == 1 && Nz == 1 && lNy >= 4 && lNy <= 12 && (size_t)z_tile_quads(lNy, film_pol(lNy), 1) * 4 * esz <= (size_t)max_smem;
}

// ---- tensor maps (TMA descriptors) for the one-request prefetch of a strided tile (kernels_v2.cuh pf_l2_tensor) --------
// 4D views of a workspace, dimension 0 = the contiguous axis in REALS (4 per quad).  The encoder is a driver function;
// it is fetched through the runtime so that the library does not link libcuda.
struct TMap { alignas(64) CUtensorMap m; };
inline bool encode_tmap4(TMap* out, size_t esz, const void* base, const unsigned long long dim[4],
                         const unsigned long long stride_bytes[3], const unsigned box[4])
{
    typedef CUresult (*Fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                           const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                           CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static Fn fn = nullptr;
    if (!fn) {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &qr) != cudaSuccess || qr != cudaDriverEntryPointSuccess || !f) {
            cudaGetLastError();
            return false;
        }
        fn = (Fn)f;
    }
    for (int i = 0; i < 4; ++i) if (box[i] < 1 || box[i] > 256 || dim[i] < 1) return false;
    if ((box[0] * esz) % 16 != 0) return false;
    for (int i = 0; i < 3; ++i) if (stride_bytes[i] % 16 != 0 || stride_bytes[i] >= (1ULL << 40)) return false;
    cuuint64_t d[4] = {dim[0], dim[1], dim[2], dim[3]}, sb[3] = {stride_bytes[0], stride_bytes[1], stride_bytes[2]};
    cuuint32_t b[4] = {box[0], box[1], box[2], box[3]}, es[4] = {1, 1, 1, 1};
    return fn(&out->m, esz == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<void*>(base), d, sb, b, es,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// ---- launchers ---------------------------------------------------------------------------------------------
template <typename T> struct Ctx {
    int sm_count;
    GeoV g;                     // y / z stages (several GPUs: hq = the pairs this rank owns)
    GeoV gx;                    // x stages (several GPUs: ny = the rows this rank owns); = g on one GPU
    GeoV gfilm;                 // one-cell-thick meshes: geometry of the fused y stage (k_z_v FILM)
    bool film;
    bool pdl = false;           // programmatic dependent launch of the five kernels (plan.cu; DEMAG_PDL; GeoV::trig = where the next grid is let in)
    bool zeo = false;           // fp32, Nz = 256 / 512: the z stage as two half-length two-pass transforms (k_z_eo_v; DEMAG_NO_ZEO)
    const CQ<T>* two = nullptr; // w_Nz^z, z < Nz/2 (k_z_eo_v)
    int z16 = 0;                // fp32, Nz = 16: the z stage in registers, two lanes per column (k_z16_v; DEMAG_NO_Z16)
    bool y32 = false;           // fp32: y schedule with a radix-32 last pass where one is instantiated (YCfg32; DEMAG_NO_Y32)
    bool ylong = true;          // long y lines (Ny >= 4096) through the staged persistent kernel (DEMAG_NO_YLONG, read at plan creation)
    int lLc, lNy, lNz;
    TwSet<T> twx, twy, twz;
    const CQ<T>* twpost;
    TMap tm_z = {}, tm_xi = {}; // W2v as the z kernel tiles it / W1v as the x C2R kernel tiles it (valid iff tm_z_nq > 0 / tm_xi_ok)
    int tm_z_nq = 0;            // pair planes per slab the W2v map was encoded for (its component stride)
    bool tm_xi_ok = false;
    const int* yslot = nullptr; // slot | mirrored << 31 of every W2v position (kernels_v2.cuh "Kv"); device memory
    // L2 prefetch distance (kernels_v2.cuh pf_l2_*): pf_waves x (co-resident blocks of the kernel), per kernel; filled
    // in at plan time (mode 0 of the launchers) from the occupancy the runtime reports
    float pf_waves = 0.f;
    mutable int pf_xf = 0, pf_xi = 0, pf_yf = 0, pf_yi = 0, pf_z = 0, pf_film = 0;
    bool sharded = false;       // several GPUs: x R2C stores through m_in, y inverse through m_out (kernels_v2.cuh ShardMap)
    ShardMap<T> m_in, m_out;
};

// launch with programmatic stream serialization (kernels_v2.cuh pdl_enter): plain pointers / PODs by value
// (pdl = false: an ordinary, fully serialised launch)
template <typename... KA, typename... A>
inline void launch_pdl(bool pdl, void (*kern)(KA...), unsigned grid, unsigned block, size_t smem, cudaStream_t st, A&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    cudaLaunchKernelEx(&cfg, kern, KA(args)...);
}

// co-resident blocks of a kernel on the whole device x pf_waves -> prefetch distance in blocks
template <typename K> inline int pf_distance(float waves, int sm_count, K kern, int nt, int smem)
{
    if (waves <= 0.f) return 0;
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, nt, (size_t)smem) != cudaSuccess || occ < 1) occ = 1;
    const float d = waves * (float)occ * (float)sm_count;
    return d < 1.f ? 1 : (int)d;
}
template <typename G> inline G with_pf(G g, int pf) { g.pf = pf; return g; }
template <typename G> inline G with_pft(G g, bool on) { g.pft = on ? 1 : 0; return g; }

#define V2_CASE_X(L, KERN, ...)                                                                                     \
    case L: {                                                                                                        \
        using C = typename CfgSel<XCfg<L>, XCfgD<L>, T>::type;                                                                                           \
        constexpr int smem = x_tile_quads(L, C::POL, C::RP) * (int)sizeof(CQ<T>);                                    \
        if (mode == 0) { *err = cudaFuncSetAttribute(KERN<T, L, C::POL, C::RP, C::NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
                         *pfd = pf_distance(c.pf_waves, c.sm_count, KERN<T, L, C::POL, C::RP, C::NT>, C::NT, smem); }  \
        else launch_pdl(c.pdl, KERN<T, L, C::POL, C::RP, C::NT>, 3u * c.gx.nz * (c.gx.ny / (2 * C::RP)), C::NT, smem, st, __VA_ARGS__); \
        return true;                                                                                                 \
    }

// mode 0: set the shared-memory attribute (plan time); mode 1: launch
template <typename T>
bool x_fwd(int mode, const Ctx<T>& c, cudaStream_t st, const T* M, CQ<T>* W1, cudaError_t* err)
{
    int* pfd = &c.pf_xf;
    const GeoV gp = with_pf(c.gx, c.pf_xf);
    switch (c.lLc) {
        V2_CASE_X(4, k_x_r2c_v, gp, M, W1, c.twx, c.twpost) V2_CASE_X(5, k_x_r2c_v, gp, M, W1, c.twx, c.twpost)
        V2_CASE_X(6, k_x_r2c_v, gp, M, W1, c.twx, c.twpost) V2_CASE_X(7, k_x_r2c_v, gp, M, W1, c.twx, c.twpost)
        V2_CASE_X(8, k_x_r2c_v, gp, M, W1, c.twx, c.twpost) V2_CASE_X(9, k_x_r2c_v, gp, M, W1, c.twx, c.twpost)
        V2_CASE_X(10, k_x_r2c_v, gp, M, W1, c.twx, c.twpost) V2_CASE_X(11, k_x_r2c_v, gp, M, W1, c.twx, c.twpost)
        V2_CASE_X(12, k_x_r2c_v, gp, M, W1, c.twx, c.twpost)
    case 13: if constexpr (sizeof(T) == 4) { switch (13) { V2_CASE_X(13, k_x_r2c_v, gp, M, W1, c.twx, c.twpost) } } return false;
    default: return false;
    }
}
// the same for an embedded caller array (kernels_v2.cuh GeoV::onx)
template <typename T>
bool x_fwd_e(int mode, const Ctx<T>& c, cudaStream_t st, const T* M, CQ<T>* W1, cudaError_t* err)
{
    int* pfd = &c.pf_xf;
    const GeoV gp = with_pf(c.gx, c.pf_xf);
    switch (c.lLc) {
        V2_CASE_X(4, k_x_r2c_e_v, gp, M, W1, c.twx, c.twpost) V2_CASE_X(5, k_x_r2c_e_v, gp, M, W1, c.twx, c.twpost)
        V2_CASE_X(6, k_x_r2c_e_v, gp, M, W1, c.twx, c.twpost) V2_CASE_X(7, k_x_r2c_e_v, gp, M, W1, c.twx, c.twpost)
        V2_CASE_X(8, k_x_r2c_e_v, gp, M, W1, c.twx, c.twpost) V2_CASE_X(9, k_x_r2c_e_v, gp, M, W1, c.twx, c.twpost)
        V2_CASE_X(10, k_x_r2c_e_v, gp, M, W1, c.twx, c.twpost) V2_CASE_X(11, k_x_r2c_e_v, gp, M, W1, c.twx, c.twpost)
        V2_CASE_X(12, k_x_r2c_e_v, gp, M, W1, c.twx, c.twpost)
    case 13: if constexpr (sizeof(T) == 4) { switch (13) { V2_CASE_X(13, k_x_r2c_e_v, gp, M, W1, c.twx, c.twpost) } } return false;
    default: return false;
    }
}
// several GPUs: rows of this rank in, pairs stored at their owners (k_x_r2c_sh_v)
template <typename T>
bool x_fwd_sh(int mode, const Ctx<T>& c, cudaStream_t st, const T* M, cudaError_t* err)
{
    int pf_unused = 0; int* pfd = &pf_unused;          // the partitioned variant does not prefetch
    switch (c.lLc) {
        V2_CASE_X(4, k_x_r2c_sh_v, c.gx, M, c.m_in, c.twx, c.twpost) V2_CASE_X(5, k_x_r2c_sh_v, c.gx, M, c.m_in, c.twx, c.twpost)
        V2_CASE_X(6, k_x_r2c_sh_v, c.gx, M, c.m_in, c.twx, c.twpost) V2_CASE_X(7, k_x_r2c_sh_v, c.gx, M, c.m_in, c.twx, c.twpost)
        V2_CASE_X(8, k_x_r2c_sh_v, c.gx, M, c.m_in, c.twx, c.twpost) V2_CASE_X(9, k_x_r2c_sh_v, c.gx, M, c.m_in, c.twx, c.twpost)
        V2_CASE_X(10, k_x_r2c_sh_v, c.gx, M, c.m_in, c.twx, c.twpost) V2_CASE_X(11, k_x_r2c_sh_v, c.gx, M, c.m_in, c.twx, c.twpost)
        V2_CASE_X(12, k_x_r2c_sh_v, c.gx, M, c.m_in, c.twx, c.twpost)
    case 13: if constexpr (sizeof(T) == 4) { switch (13) { V2_CASE_X(13, k_x_r2c_sh_v, c.gx, M, c.m_in, c.twx, c.twpost) } } return false;
    default: return false;
    }
}
template <typename T>
bool x_inv(int mode, const Ctx<T>& c, cudaStream_t st, const CQ<T>* W1, T* H, cudaError_t* err, int acc = 0)
{
    int* pfd = &c.pf_xi;
    GeoV ga = c.gx; ga.acc = acc; ga.pf = c.pf_xi; ga.pft = c.tm_xi_ok ? 1 : 0;
    switch (c.lLc) {
        V2_CASE_X(4, k_x_c2r_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m) V2_CASE_X(5, k_x_c2r_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m)
        V2_CASE_X(6, k_x_c2r_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m) V2_CASE_X(7, k_x_c2r_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m)
        V2_CASE_X(8, k_x_c2r_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m) V2_CASE_X(9, k_x_c2r_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m)
        V2_CASE_X(10, k_x_c2r_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m) V2_CASE_X(11, k_x_c2r_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m)
        V2_CASE_X(12, k_x_c2r_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m)
    case 13: if constexpr (sizeof(T) == 4) { switch (13) { V2_CASE_X(13, k_x_c2r_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m) } } return false;
    default: return false;
    }
}

template <typename T>
bool x_inv_e(int mode, const Ctx<T>& c, cudaStream_t st, const CQ<T>* W1, T* H, cudaError_t* err, int acc = 0)
{
    int* pfd = &c.pf_xi;
    GeoV ga = c.gx; ga.acc = acc; ga.pf = c.pf_xi; ga.pft = c.tm_xi_ok ? 1 : 0;
    switch (c.lLc) {
        V2_CASE_X(4, k_x_c2r_e_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m) V2_CASE_X(5, k_x_c2r_e_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m)
        V2_CASE_X(6, k_x_c2r_e_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m) V2_CASE_X(7, k_x_c2r_e_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m)
        V2_CASE_X(8, k_x_c2r_e_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m) V2_CASE_X(9, k_x_c2r_e_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m)
        V2_CASE_X(10, k_x_c2r_e_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m) V2_CASE_X(11, k_x_c2r_e_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m)
        V2_CASE_X(12, k_x_c2r_e_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m)
    case 13: if constexpr (sizeof(T) == 4) { switch (13) { V2_CASE_X(13, k_x_c2r_e_v, ga, W1, H, c.twx, c.twpost, c.tm_xi.m) } } return false;
    default: return false;
    }
}

#define V2_CASE_Y(L, KERN, A, B) case L: V2_BODY_Y(L, KERN, A, B)
#define V2_BODY_Y(L, KERN, A, B) V2_BODY_Y_C(typename CfgSel<YCfg<L> COMMA YCfgD<L> COMMA T>::type, L, KERN, A, B)
#define V2_BODY_Y_C(CFG, L, KERN, A, B)                                                                             \
    {                                                                                                                \
        using C = CFG;                                                                                               \
        constexpr int smem = y_tile_quads(L, C::POL, C::BP) * (int)sizeof(CQ<T>);                                    \
        if (mode == 0) { *err = cudaFuncSetAttribute(KERN<T, L, C::POL, C::BP, C::NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
                         *pfd = pf_distance(c.pf_waves, c.sm_count, KERN<T, L, C::POL, C::BP, C::NT>, C::NT, smem); }  \
        else launch_pdl(c.pdl, KERN<T, L, C::POL, C::BP, C::NT>, (unsigned)((3LL * nq * c.g.nz + C::BP - 1) / C::BP), C::NT, smem, st, with_pf(c.g, *pfd), q0, nq, A, B, c.twy); \
        return true;                                                                                                 \
    }
#define COMMA ,
#define V2_BODY_YLONG(L) V2_BODY_YLONG_C(typename CfgSel<YCfg<L> COMMA YCfgD<L> COMMA T>::type, L)
#define V2_BODY_YLONG_C(CFG, L)                                                                                     \
    {                                                                                                                \
        using C = CFG;                                                                                               \
        constexpr int smem = (y_tile_quads(L, C::POL, 1) + (1 << (L - 1))) * (int)sizeof(CQ<T>);                      \
        if (mode == 0) *err = cudaFuncSetAttribute(k_y_fwd_long_v<T, L, C::POL, C::NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
        else { const long long nl = 3LL * nq * c.g.nz;                                                               \
               launch_pdl(c.pdl, k_y_fwd_long_v<T, L, C::POL, C::NT>, (unsigned)(nl < c.sm_count ? nl : c.sm_count), C::NT, smem, st, c.g, q0, nq, W1, W2, c.twy); } \
        return true;                                                                                                 \
    }
template <typename T>
bool y_fwd(int mode, const Ctx<T>& c, cudaStream_t st, int q0, int nq, const CQ<T>* W1, CQ<T>* W2, cudaError_t* err)
{
    int* pfd = &c.pf_yf;
    if constexpr (sizeof(T) == 4) {
        if (c.y32 && c.lNy == 9) V2_BODY_Y_C(YCfg32<9>, 9, k_y_fwd_v, W1, W2)
        if (c.y32 && c.lNy == 13 && c.ylong) V2_BODY_YLONG_C(YCfg32<13>, 13)
        if (c.y32 && c.lNy == 13) V2_BODY_Y_C(YCfg32<13>, 13, k_y_fwd_v, W1, W2)
    }
    if (c.lNy == 12 && c.ylong) V2_BODY_YLONG(12)
    if constexpr (sizeof(T) == 4) { if (c.lNy == 13 && c.ylong) V2_BODY_YLONG(13) }
    switch (c.lNy) {
        V2_CASE_Y(4, k_y_fwd_v, W1, W2) V2_CASE_Y(5, k_y_fwd_v, W1, W2) V2_CASE_Y(6, k_y_fwd_v, W1, W2) V2_CASE_Y(7, k_y_fwd_v, W1, W2)
        V2_CASE_Y(8, k_y_fwd_v, W1, W2) V2_CASE_Y(9, k_y_fwd_v, W1, W2) V2_CASE_Y(10, k_y_fwd_v, W1, W2) V2_CASE_Y(11, k_y_fwd_v, W1, W2)
        V2_CASE_Y(12, k_y_fwd_v, W1, W2)
    case 13: if constexpr (sizeof(T) == 4) V2_BODY_Y(13, k_y_fwd_v, W1, W2) else return false;
    default: return false;
    }
}
template <typename T>
bool y_inv(int mode, const Ctx<T>& c, cudaStream_t st, int q0, int nq, const CQ<T>* W2, CQ<T>* W1, cudaError_t* err)
{
    int* pfd = &c.pf_yi;
    if constexpr (sizeof(T) == 4) {
        if (c.y32 && c.lNy == 9) V2_BODY_Y_C(YCfg32<9>, 9, k_y_inv_v, W2, W1)
        if (c.y32 && c.lNy == 13) V2_BODY_Y_C(YCfg32<13>, 13, k_y_inv_v, W2, W1)
    }
    switch (c.lNy) {
        V2_CASE_Y(4, k_y_inv_v, W2, W1) V2_CASE_Y(5, k_y_inv_v, W2, W1) V2_CASE_Y(6, k_y_inv_v, W2, W1) V2_CASE_Y(7, k_y_inv_v, W2, W1)
        V2_CASE_Y(8, k_y_inv_v, W2, W1) V2_CASE_Y(9, k_y_inv_v, W2, W1) V2_CASE_Y(10, k_y_inv_v, W2, W1) V2_CASE_Y(11, k_y_inv_v, W2, W1)
        V2_CASE_Y(12, k_y_inv_v, W2, W1)
    case 13: if constexpr (sizeof(T) == 4) V2_BODY_Y(13, k_y_inv_v, W2, W1) else return false;
    default: return false;
    }
}

// several GPUs: the cropped rows stored at the ranks that own them (k_y_inv_sh_v)
#define V2_CASE_YSH(L) case L: V2_BODY_YSH_C(typename CfgSel<YCfg<L> COMMA YCfgD<L> COMMA T>::type, L)
#define V2_BODY_YSH_C(CFG, L)                                                                                       \
    {                                                                                                                \
        using C = CFG;                                                                                               \
        constexpr int smem = y_tile_quads(L, C::POL, C::BP) * (int)sizeof(CQ<T>);                                    \
        if (mode == 0) *err = cudaFuncSetAttribute(k_y_inv_sh_v<T, L, C::POL, C::BP, C::NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
        else k_y_inv_sh_v<T, L, C::POL, C::BP, C::NT><<<(unsigned)((3LL * nq * c.g.nz + C::BP - 1) / C::BP), C::NT, smem, st>>>(c.g, q0, nq, W2, c.m_out, c.twy); \
        return true;                                                                                                 \
    }
template <typename T>
bool y_inv_sh(int mode, const Ctx<T>& c, cudaStream_t st, int q0, int nq, const CQ<T>* W2, cudaError_t* err)
{
    if constexpr (sizeof(T) == 4) {
        if (c.y32 && c.lNy == 9) V2_BODY_YSH_C(YCfg32<9>, 9)
        if (c.y32 && c.lNy == 13) V2_BODY_YSH_C(YCfg32<13>, 13)
    }
    switch (c.lNy) {
        V2_CASE_YSH(4) V2_CASE_YSH(5) V2_CASE_YSH(6) V2_CASE_YSH(7) V2_CASE_YSH(8) V2_CASE_YSH(9) V2_CASE_YSH(10) V2_CASE_YSH(11)
        V2_CASE_YSH(12)
    case 13: if constexpr (sizeof(T) == 4) { switch (13) { V2_CASE_YSH(13) } } return false;
    default: return false;
    }
}

#define V2_CASE_Z(L)                                                                                                \
    case L: {                                                                                                        \
        using C = typename CfgSel<ZCfg<L>, ZCfgD<L>, T>::type;                                                                                           \
        constexpr int smem = z_tile_quads(L, C::POL, C::TY) * (int)sizeof(CQ<T>);                                    \
        if (mode == 0) { *err = cudaFuncSetAttribute(k_z_v<T, L, C::POL, C::TY, C::NT, C::MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
                         c.pf_z = pf_distance(c.pf_waves, c.sm_count, k_z_v<T, L, C::POL, C::TY, C::NT, C::MINB>, C::NT, smem); } \
        else launch_pdl(c.pdl, k_z_v<T, L, C::POL, C::TY, C::NT, C::MINB>, (unsigned)(nq * (c.g.Ny / C::TY)), C::NT, smem, st, with_pft(with_pf(c.g, c.pf_z), nq == c.tm_z_nq), q0, nq, W2, K, c.yslot, c.twz, c.tm_z.m); \
        return true;                                                                                                 \
    }
template <typename T>
bool z_mul(int mode, const Ctx<T>& c, cudaStream_t st, int q0, int nq, CQ<T>* W2, const typename kchunks<T>::V* K, cudaError_t* err)
{
    if constexpr (sizeof(T) == 4) {
        if (c.lNz == 4 && c.z16 && c.g.Ny % 64 == 0) {
            if (mode && c.z16 == 2) launch_pdl(c.pdl, k_z16_v<T, 2>, (unsigned)(nq * (c.g.Ny / 64)), 128, 0, st, with_pf(c.g, c.pf_z), q0, nq, W2, K, c.yslot);
            else if (mode) launch_pdl(c.pdl, k_z16_v<T, 3>, (unsigned)(nq * (c.g.Ny / 64)), 128, 0, st, with_pf(c.g, c.pf_z), q0, nq, W2, K, c.yslot);
            else c.pf_z = c.pf_waves > 0.f ? 1 : 0;
            return true;
        }
    }
    if constexpr (sizeof(T) == 4) {
#define V2_ZEO(L, TY_, NT_)                                                                                           \
        {                                                                                                            \
            constexpr int smem = ((1 << L) * 3 * TY_ + TY_) * (int)sizeof(CQ<T>);                                    \
            if (mode == 0) { *err = cudaFuncSetAttribute(k_z_eo_v<T, L, TY_, NT_>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
                             c.pf_z = pf_distance(c.pf_waves, c.sm_count, k_z_eo_v<T, L, TY_, NT_>, NT_, smem); }    \
            else launch_pdl(c.pdl, k_z_eo_v<T, L, TY_, NT_>, (unsigned)(nq * (c.g.Ny / TY_)), NT_, smem, st,          \
                            with_pft(with_pf(c.g, c.pf_z), nq == c.tm_z_nq), q0, nq, W2, K, c.yslot, c.twz, c.two, c.tm_z.m); \
            return true;                                                                                             \
        }
        if (c.zeo && c.lNz == 9) V2_ZEO(9, 4, 128)
        if (c.zeo && c.lNz == 8) V2_ZEO(8, 4, 64)
    }
    switch (c.lNz) {
    case 0: if (mode) launch_pdl(c.pdl, k_z1_v<T, 0>, (unsigned)(nq * (c.g.Ny / (c.g.Ny < 128 ? c.g.Ny : 128))), c.g.Ny < 128 ? c.g.Ny : 128, 0, st, c.g, q0, nq, W2, K, c.yslot); return true;
    case 2: if (mode) launch_pdl(c.pdl, k_z1_v<T, 2>, (unsigned)(nq * (c.g.Ny / (c.g.Ny < 128 ? c.g.Ny : 128))), c.g.Ny < 128 ? c.g.Ny : 128, 0, st, c.g, q0, nq, W2, K, c.yslot); return true;
    case 3: if (mode) launch_pdl(c.pdl, k_z1_v<T, 3>, (unsigned)(nq * (c.g.Ny / (c.g.Ny < 128 ? c.g.Ny : 128))), c.g.Ny < 128 ? c.g.Ny : 128, 0, st, c.g, q0, nq, W2, K, c.yslot); return true;
        V2_CASE_Z(4) V2_CASE_Z(5) V2_CASE_Z(6) V2_CASE_Z(7) V2_CASE_Z(8) V2_CASE_Z(9) V2_CASE_Z(10) V2_CASE_Z(11)
    default: return false;
    }
}

// fused y stage of a one-cell-thick mesh: k_z_v<FILM> along y, in place on W1v
#define V2_CASE_FILM(L, POL_, NT_)                                                                                  \
    case L: {                                                                                                        \
        constexpr int smem = z_tile_quads(L, POL_, 1) * (int)sizeof(CQ<T>);                                          \
        if (mode == 0) { *err = cudaFuncSetAttribute(k_z_v<T, L, POL_, 1, NT_, 1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
                         c.pf_film = pf_distance(c.pf_waves, c.sm_count, k_z_v<T, L, POL_, 1, NT_, 1, true>, NT_, smem); } \
        else launch_pdl(c.pdl, k_z_v<T, L, POL_, 1, NT_, 1, true>, (unsigned)c.g.hq, NT_, smem, st, with_pf(c.gfilm, c.pf_film), 0, c.g.hq, W1, K, (const int*)nullptr, c.twy, c.tm_z.m); \
        return true;                                                                                                 \
    }
template <typename T>
bool y_film(int mode, const Ctx<T>& c, cudaStream_t st, CQ<T>* W1, const typename kchunks<T>::V* K, cudaError_t* err)
{
    switch (c.lNy) {
        V2_CASE_FILM(4, 0, 32) V2_CASE_FILM(5, 1, 32) V2_CASE_FILM(6, 1, 32) V2_CASE_FILM(7, 1, 32) V2_CASE_FILM(8, 2, 64)
        V2_CASE_FILM(9, 1, 64) V2_CASE_FILM(10, 1, 128) V2_CASE_FILM(11, 2, 256) V2_CASE_FILM(12, 1, 512)
    default: return false;
    }
}

}  // namespace v2
}  // namespace demag
