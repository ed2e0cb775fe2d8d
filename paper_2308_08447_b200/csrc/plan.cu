// plan.cu -- the C ABI of include/demag.h: argument checking, workspace, launch configuration.
// Every step of the hot path runs in the kernels of kernels.cuh; this file only enqueues them.
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <algorithm>
#include <new>
#include <vector>

#include "../../include/demag.h"
#include "builder.cuh"
#include "kernels.cuh"
#include "kernels_z.cuh"
#include "v2_host.cuh"

// The fast-path launchers are instantiated in their own translation units (v2_inst.cuh: one per stage and precision),
// so that the library builds in parallel.
namespace demag {
namespace v2 {
#define V2_EXTERN(T)                                                                                                      \
    extern template bool x_fwd<T>(int, const Ctx<T>&, cudaStream_t, const T*, CQ<T>*, cudaError_t*);                     \
    extern template bool x_fwd_sh<T>(int, const Ctx<T>&, cudaStream_t, const T*, cudaError_t*);                          \
    extern template bool x_inv<T>(int, const Ctx<T>&, cudaStream_t, const CQ<T>*, T*, cudaError_t*, int);                \
    extern template bool x_fwd_e<T>(int, const Ctx<T>&, cudaStream_t, const T*, CQ<T>*, cudaError_t*);                   \
    extern template bool x_inv_e<T>(int, const Ctx<T>&, cudaStream_t, const CQ<T>*, T*, cudaError_t*, int);              \
    extern template bool y_fwd<T>(int, const Ctx<T>&, cudaStream_t, int, int, const CQ<T>*, CQ<T>*, cudaError_t*);       \
    extern template bool y_inv<T>(int, const Ctx<T>&, cudaStream_t, int, int, const CQ<T>*, CQ<T>*, cudaError_t*);       \
    extern template bool y_inv_sh<T>(int, const Ctx<T>&, cudaStream_t, int, int, const CQ<T>*, cudaError_t*);            \
    extern template bool z_mul<T>(int, const Ctx<T>&, cudaStream_t, int, int, CQ<T>*, const typename kchunks<T>::V*, cudaError_t*); \
    extern template bool y_film<T>(int, const Ctx<T>&, cudaStream_t, CQ<T>*, const typename kchunks<T>::V*, cudaError_t*);
V2_EXTERN(float)
V2_EXTERN(double)
#undef V2_EXTERN
}  // namespace v2
}  // namespace demag

using namespace demag;

namespace {

thread_local char g_err[512] = "";

demag_status fail(demag_status st, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return st;
}

#define CUDA_TRY(call)                                                                          \
    do {                                                                                        \
        cudaError_t e_ = (call);                                                                \
        if (e_ != cudaSuccess)                                                                  \
            return fail(e_ == cudaErrorMemoryAllocation ? DEMAG_ERR_ALLOC : DEMAG_ERR_CUDA,     \
                        "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__);   \
    } while (0)

constexpr int kMaxSmem = 232448 - 1024;   // 227 KB opt-in shared memory per CTA (sm_100) minus room for static __shared__
constexpr size_t kSlabBytes = (size_t)16 << 30;   // cap of the W2 workspace: larger meshes run the y/z stages slab by slab.
                                                  // (Measured on B200: the kernels are not DRAM bound, an L2-sized slab only adds launches and
                                                  //  partial waves -- C3 426 us at 128 MB vs 401 us unslabbed -- so the cap is a memory cap.)

inline bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }
inline int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }
inline int pow2_floor(long long v) { int p = 1; while (2LL * p <= v) p *= 2; return p; }
inline int pow2_ceil(int v) { int p = 1; while (p < v) p *= 2; return p; }

}  // namespace

struct demag_plan_s {
    Geo g;
    double h[3];
    unsigned pbc;
    int pbc_images = 10;   // built-in periodic tensor: images summed on each side of a periodic axis (demag_set_pbc_images)
    int prec;
    size_t esz;       // sizeof real
    int device;
    int sm_count;
    void* W1 = nullptr; size_t w1_bytes = 0;
    void* W2 = nullptr; size_t w2_bytes = 0;
    void* K = nullptr;  size_t k_bytes = 0, kcomp_stride = 0;
    void* tw[3] = {nullptr, nullptr, nullptr}; size_t tw_bytes = 0;
    void* Mc = nullptr; void* Hc = nullptr; size_t macro_bytes = 0;   // atomistic macrocell buffers
    bool has_kernel = false;
    // launch configuration
    int R1, thr1, smem1, pitch1;  // K1 / K5   (pitch odd -> conflict-free transposing loads; B == 1 -> swizzle)
    int B2, thr2, smem2, pitch2;  // K2 / K4
    int TY, thr3, smem3;          // K3
    int nkx_slab, nkx_auto;
    bool fast1 = false, fast2 = false;   // kernels_fast.cuh variants of the x / y stages
    bool z_spec = false;                 // kernels_z.cuh compile-time specialised z stage
    // fast path (kernels_v2.cuh): pair layout of W1 / W2 / K, per-pass twiddle tables
    bool v2 = false;
    int nq_slab = 0, nq_auto = 0;        // (k, Lc-k) pair planes per L2-resident slab
    v2::Ctx<float> cf; v2::Ctx<double> cd;
    v2::AxisTables<float> tf[3]; v2::AxisTables<double> td[3];
    int* ypos2freq = nullptr;
    int* yslot = nullptr;                // fast path: slot | mirrored << 31 of every W2v position (y-packed kernel spectrum)
    int kpitch_v = 1;
    // general mesh sizes: the caller's mesh on[] is embedded (zeros) in the power-of-two mesh g.n* the transforms run on
    int on[3] = {0, 0, 0};
    bool embed = false;
    bool embed_fused = false;            // fast path, even caller nx: the x kernels read M / write H of the caller directly (no copies)
    void* Mp = nullptr; void* Hp = nullptr;
    // several GPUs (demag_plan_create_sharded): W1 is W1in [3][nq_loc][nz][ny], W1out is [3][hq][nz][ny_loc]
    bool sharded = false, peers_set = false;
    int world = 1, rank = 0, y0 = 0, ny_loc = 0, q0 = 0, nq_loc = 0;
    void* W1out = nullptr; size_t w1out_bytes = 0;
    void* ipc_open[2 * v2::kMaxRanks] = {};
};

namespace {

int pick_threads(long long elems)
{
    long long t = elems / 16;
    t = (t + 31) / 32 * 32;
    if (t < 64) t = 64;
    if (t > 512) t = 512;
    return (int)t;
}

template <typename T>
demag_status set_func_attrs()
{
    CUDA_TRY(cudaFuncSetAttribute(k_x_r2c<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
    CUDA_TRY(cudaFuncSetAttribute(k_x_c2r<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
    CUDA_TRY(cudaFuncSetAttribute(k_y_fwd<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
    CUDA_TRY(cudaFuncSetAttribute(k_y_inv<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
    CUDA_TRY(cudaFuncSetAttribute(k_x_r2c<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
    CUDA_TRY(cudaFuncSetAttribute(k_x_c2r<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
    CUDA_TRY(cudaFuncSetAttribute(k_y_fwd<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
    CUDA_TRY(cudaFuncSetAttribute(k_y_inv<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
    CUDA_TRY(cudaFuncSetAttribute(k_x_r2c_f<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
    CUDA_TRY(cudaFuncSetAttribute(k_x_c2r_f<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
    CUDA_TRY(cudaFuncSetAttribute(k_y_fwd_f<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
    CUDA_TRY(cudaFuncSetAttribute(k_y_inv_f<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
    CUDA_TRY(cudaFuncSetAttribute(k_z_mul<T, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
    CUDA_TRY(cudaFuncSetAttribute(k_z_mul<T, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
    CUDA_TRY(cudaFuncSetAttribute(k_z_mul<T, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
    return DEMAG_OK;
}

// exp(-2 pi i k / N), k = 0..N-1, evaluated in long double, octant-reduced
template <typename C>
demag_status make_twiddles(int N, void** out, size_t* bytes)
{
    std::vector<C> t((size_t)N);
    const long double tp = 6.283185307179586476925286766559005768L;
    for (int k = 0; k < N; ++k) {
        const long double a = tp * (long double)k / (long double)N;
        t[k].x = (decltype(C::x))cosl(a);
        t[k].y = (decltype(C::x))(-sinl(a));
    }
    if (N >= 4) { t[N / 4].x = 0; t[N / 4].y = -1; t[N / 2].x = -1; t[N / 2].y = 0; t[3 * N / 4].x = 0; t[3 * N / 4].y = 1; }
    else if (N == 2) { t[1].x = -1; t[1].y = 0; }
    CUDA_TRY(cudaMalloc(out, sizeof(C) * (size_t)N));
    CUDA_TRY(cudaMemcpy(*out, t.data(), sizeof(C) * (size_t)N, cudaMemcpyHostToDevice));
    *bytes += sizeof(C) * (size_t)N;
    return DEMAG_OK;
}

// Compile-time specialised z stage (kernels_z.cuh) for (log2 Nz, TY) in {(4..8, 16), (9, 8)}.
// mode 0: set the shared-memory attribute (plan time); mode 1: launch.  Returns false if no specialisation matches.
template <typename T, int LNZ, int TY, int NT>
bool z_c_do(int mode, const Geo& g, unsigned grid, cudaStream_t st, int kx0, int nkx, typename cx_of<T>::type* W2,
            const T* K, size_t kcs, const typename cx_of<T>::type* twz, cudaError_t* err)
{
    constexpr int smem = (1 << LNZ) * 3 * TY * (int)sizeof(typename cx_of<T>::type);
    if (mode == 0) *err = cudaFuncSetAttribute(k_z_mul_c<T, LNZ, TY, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    else k_z_mul_c<T, LNZ, TY, NT><<<grid, NT, smem, st>>>(g, kx0, nkx, W2, K, kcs, twz);
    return true;
}
template <typename T>
bool z_c_dispatch(int mode, const Geo& g, int TY, unsigned grid, cudaStream_t st, int kx0, int nkx,
                  typename cx_of<T>::type* W2, const T* K, size_t kcs, const typename cx_of<T>::type* twz, cudaError_t* err)
{
    if (TY == 16) {
        switch (g.lNz) {
        case 4: return z_c_do<T, 4, 16, 96>(mode, g, grid, st, kx0, nkx, W2, K, kcs, twz, err);
        case 5: return z_c_do<T, 5, 16, 192>(mode, g, grid, st, kx0, nkx, W2, K, kcs, twz, err);
        case 6: return z_c_do<T, 6, 16, 384>(mode, g, grid, st, kx0, nkx, W2, K, kcs, twz, err);
        case 7: return z_c_do<T, 7, 16, 384>(mode, g, grid, st, kx0, nkx, W2, K, kcs, twz, err);
        case 8: if (sizeof(T) == 4) return z_c_do<T, 8, 16, 384>(mode, g, grid, st, kx0, nkx, W2, K, kcs, twz, err); break;
        default: break;
        }
    } else if (TY == 8) {
        if (g.lNz == 9 && sizeof(T) == 4) return z_c_do<T, 9, 8, 384>(mode, g, grid, st, kx0, nkx, W2, K, kcs, twz, err);
        if (g.lNz == 8 && sizeof(T) == 8) return z_c_do<T, 8, 8, 384>(mode, g, grid, st, kx0, nkx, W2, K, kcs, twz, err);
    }
    return false;
}

void configure(demag_plan_s* p)
{
    const Geo& g = p->g;
    const size_t csz = 2 * p->esz;
    // K1 / K5: R rows of Lc complex, tile s[Lc][pitch].  R >= 4 keeps the transposed stores at >= 32 B runs.
    {
        const long long Lc = 1LL << g.lLc;
        int R = pow2_floor(std::max<long long>(1, (48 << 10) / (long long)(Lc * csz)));
        if (R < 4) R = 4;
        if (R > 16) R = 16;
        while (R > 1 && (long long)(R | 1) * Lc * csz > 200 << 10) R /= 2;
        if (R > g.ny) R = g.ny;
        p->R1 = R;
        p->pitch1 = R == 1 ? 1 : (R | 1);
        p->fast1 = g.lLc >= 3 && R >= 2;
        const long long elems = (long long)p->pitch1 * Lc;
        p->smem1 = (int)(((elems + 15) / 16 * 16) * csz);
        p->thr1 = pick_threads((long long)R * Lc);
    }
    // K2 / K4: B lines of Ny complex, tile s[Ny][pitch]: the largest B in {16,8,4,2} whose tile is <= 100 KB
    {
        int B = 16;
        long long lim = 100 << 10;
        if (const char* e = getenv("DEMAG_B2_KB")) { const int v = atoi(e); if (v >= 1 && v <= 220) lim = (long long)v << 10; }   // tuning override
        while (B > 1 && (long long)(B | 1) * g.Ny * csz > lim) B /= 2;
        const long long nlines_min = 3LL * g.nz;
        while (B > nlines_min) B /= 2;
        if (B < 1) B = 1;
        p->B2 = B;
        p->pitch2 = B == 1 ? 1 : (B | 1);
        p->fast2 = g.lNy >= 3 && B >= 2;
        const long long elems = (long long)p->pitch2 * g.Ny;
        p->smem2 = (int)(((elems + 15) / 16 * 16) * csz);
        p->thr2 = pick_threads((long long)B * g.Ny);
    }
    // K3: TY ky columns x Nz x 3 components, tile s[Nz][3*TY]; block = a multiple of 3*TY threads
    if (g.lNz <= 3) {                       // whole z transform in one butterfly per thread, no shared memory
        int TY = std::min(g.Ny, 128);
        p->TY = TY; p->smem3 = 0; p->thr3 = std::max(32, TY);
    } else {
        int TY = 16;
        if (const char* e = getenv("DEMAG_TY")) { const int v = atoi(e); if (v >= 1 && v <= 64 && is_pow2(v)) TY = v; }   // tuning override (experiments only)
        while (TY > 1 && (long long)TY * 3 * g.Nz * csz > 100 << 10) TY /= 2;
        if (TY > g.Ny) TY = g.Ny;
        p->TY = TY;
        const int B = 3 * TY;
        p->smem3 = (int)((long long)B * g.Nz * csz);
        const int S0 = g.Nz / 8;
        const int gc = pow2_floor(std::max(1, std::min(S0, 512 / B)));
        p->thr3 = B * gc;
    }
    // slab of kx planes whose W2 part stays L2-resident between K2, K3 and K4
    {
        const size_t per_kx = (size_t)3 * g.nz * g.Ny * csz;
        size_t slab_bytes = kSlabBytes;
        if (const char* e = getenv("DEMAG_SLAB_MB")) { const long long v = atoll(e); if (v >= 1 && v <= (1LL << 20)) slab_bytes = (size_t)v << 20; }   // tuning override
        long long n = (long long)(slab_bytes / per_kx);
        if (n < 1) n = 1;
        if (n > g.hx) n = g.hx;
        p->nkx_auto = (int)n;
        p->nkx_slab = (int)n;
    }
}

}  // namespace

extern "C" {

const char* demag_last_error(void) { return g_err; }

static demag_status plan_create_impl(demag_plan_t* out, int nx, int ny, int nz, double hx, double hy, double hz,
                                     unsigned pbc_flags, int precision, int rank, int world, bool sharded);

demag_status demag_plan_create(demag_plan_t* out, int nx, int ny, int nz, double hx, double hy, double hz,
                               unsigned pbc_flags, int precision)
{
    return plan_create_impl(out, nx, ny, nz, hx, hy, hz, pbc_flags, precision, 0, 1, false);
}

demag_status demag_plan_create_sharded(demag_plan_t* out, int nx, int ny, int nz, double hx, double hy, double hz,
                                       unsigned pbc_flags, int precision, int rank, int world)
{
    return plan_create_impl(out, nx, ny, nz, hx, hy, hz, pbc_flags, precision, rank, world, true);
}

demag_status demag_shard_range(int n, int world, int rank, int align, int* begin, int* count)
{
    g_err[0] = 0;
    if (n < 1 || world < 1 || rank < 0 || rank >= world || align < 1 || !begin || !count)
        return fail(DEMAG_ERR_INVALID_ARG, "demag_shard_range: bad arguments (n %d, world %d, rank %d, align %d)", n, world, rank, align);
    const int per = n / world / align * align;
    if (per == 0) return fail(DEMAG_ERR_UNSUPPORTED, "%d units cannot be split over %d ranks in multiples of %d", n, world, align);
    *begin = rank * per;
    *count = rank == world - 1 ? n - rank * per : per;
    return DEMAG_OK;
}

static demag_status plan_create_impl(demag_plan_t* out, int nx, int ny, int nz, double hx, double hy, double hz,
                                     unsigned pbc_flags, int precision, int rank, int world, bool sharded)
{
    g_err[0] = 0;
    if (!out) return fail(DEMAG_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 1) return fail(DEMAG_ERR_INVALID_ARG, "mesh sizes must be >= 1");
    if (!(hx > 0 && hy > 0 && hz > 0) || !isfinite(hx) || !isfinite(hy) || !isfinite(hz))
        return fail(DEMAG_ERR_INVALID_ARG, "cell sizes must be positive and finite");
    if (precision != DEMAG_FP32 && precision != DEMAG_FP64) return fail(DEMAG_ERR_INVALID_ARG, "bad precision");
    if (pbc_flags & ~7u) return fail(DEMAG_ERR_INVALID_ARG, "bad pbc_flags");
    // x rows up to 8192 cells (a 16384-point real transform = 8192 quads = 128 KB of shared memory: the paper's own
    // 7680 x 3840 x 2 mesh); y and z lines up to 4096 cells (an 8192-point line pair is the largest tile)
    if (nx > 8192 || ny > 4096 || nz > 4096) return fail(DEMAG_ERR_UNSUPPORTED, "mesh sizes must be <= 8192 x 4096 x 4096");
    if (((pbc_flags & DEMAG_PBC_X) && !is_pow2(nx)) || ((pbc_flags & DEMAG_PBC_Y) && !is_pow2(ny)) ||
        ((pbc_flags & DEMAG_PBC_Z) && !is_pow2(nz)))
        return fail(DEMAG_ERR_UNSUPPORTED, "a periodic axis cannot be padded: its size must be a power of two (got %d x %d x %d)", nx, ny, nz);

    if (sharded) {
        if (world < 1 || world > v2::kMaxRanks || rank < 0 || rank >= world)
            return fail(DEMAG_ERR_INVALID_ARG, "bad rank %d / world %d (1 <= world <= %d)", rank, world, v2::kMaxRanks);
        if (!is_pow2(nx) || !is_pow2(ny) || !is_pow2(nz) || nz < 2 || pbc_flags)
            return fail(DEMAG_ERR_UNSUPPORTED, "a sharded plan needs power-of-two mesh sizes, nz >= 2 and no periodic axis");
    }
    demag_plan_s* p = new (std::nothrow) demag_plan_s();
    if (!p) return fail(DEMAG_ERR_ALLOC, "out of host memory");
    p->sharded = sharded; p->world = world; p->rank = rank;
    // General sizes (R10): the transforms need power-of-two lengths N_a >= 2 n_a - 1 for an exact linear
    // convolution, so the mesh is embedded, with zeros, in the mesh of the next powers of two.
    p->on[0] = nx; p->on[1] = ny; p->on[2] = nz;
    nx = pow2_ceil(nx); ny = pow2_ceil(ny); nz = pow2_ceil(nz);
    p->embed = nx != p->on[0] || ny != p->on[1] || nz != p->on[2];
    Geo& g = p->g;
    g.nx = nx; g.ny = ny; g.nz = nz;
    g.Nx = (nx == 1 || (pbc_flags & DEMAG_PBC_X)) ? nx : 2 * nx;
    g.Ny = (ny == 1 || (pbc_flags & DEMAG_PBC_Y)) ? ny : 2 * ny;
    g.Nz = (nz == 1 || (pbc_flags & DEMAG_PBC_Z)) ? nz : 2 * nz;
    g.hx = g.Nx / 2 + 1;
    g.lLc = g.Nx >= 2 ? ilog2(g.Nx / 2) : 0;
    g.lNy = ilog2(g.Ny); g.lNz = ilog2(g.Nz);
    g.kpy = g.Ny / 2 + 1; g.kpz = g.Nz / 2 + 1;
    g.kpitch = g.Ny;                          // kernel rows: y unpacked, position order
    p->h[0] = hx; p->h[1] = hy; p->h[2] = hz;
    p->pbc = pbc_flags; p->prec = precision;
    p->esz = precision == DEMAG_FP32 ? 4 : 8;
    demag_status st = DEMAG_OK;
    cudaError_t e = cudaGetDevice(&p->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, p->device);
    if (e != cudaSuccess) { delete p; return fail(DEMAG_ERR_CUDA, "no CUDA device: %s", cudaGetErrorString(e)); }
    configure(p);
    const size_t csz = 2 * p->esz;
    p->w1_bytes = (size_t)3 * g.hx * g.nz * g.ny * csz;
    p->w2_bytes = (size_t)3 * p->nkx_auto * g.nz * g.Ny * csz;
    p->kcomp_stride = (size_t)g.hx * g.kpz * g.kpitch;
    p->k_bytes = 6 * p->kcomp_stride * p->esz;
    {
        const char* path = getenv("DEMAG_PATH");           // "generic" forces the size-generic kernels (tests, A/B timing)
        // fp64: the 32-byte quads halve the shared-memory efficiency of the y stage; the generic kernels are faster
        // there (C3 fp64: 1.14 ms vs 1.28 ms), so the fast family is opt-in (DEMAG_PATH=fast) for fp64 plans
        const bool want = precision == DEMAG_FP32 || (path && !strcmp(path, "fast"));
        p->v2 = want && !(path && !strcmp(path, "generic")) && pbc_flags == 0 &&
                v2::supported(nx, ny, nz, g.Nx, g.Ny, g.Nz, g.lLc, g.lNy, g.lNz, p->esz, kMaxSmem);
    }
    if (!p->v2 && (p->smem1 > kMaxSmem || p->smem2 > kMaxSmem || p->smem3 > kMaxSmem)) {
        const int worst = std::max(p->smem1, std::max(p->smem2, p->smem3));
        delete p;
        return fail(DEMAG_ERR_UNSUPPORTED, "a transform line of this plan needs %d bytes of shared memory (limit %d): "
                    "8192-point z lines are fp32 only", worst, kMaxSmem);
    }
    if (sharded && !p->v2) {
        delete p;
        return fail(DEMAG_ERR_UNSUPPORTED, "a sharded plan needs the fast kernel family (sizes in its range; DEMAG_PATH=fast for fp64)");
    }
    if (p->v2) {
        v2::GeoV gv;
        gv.nx = nx; gv.ny = ny; gv.nz = nz; gv.Ny = g.Ny; gv.Nz = g.Nz; gv.Lc = nx; gv.hq = nx / 2 + 1; gv.kpz = g.kpz; gv.acc = 0; gv.trig = 0; gv.pf = 0; gv.pft = 0; gv.onx = nx; gv.ony = ny; gv.onz = nz; gv.kst = (g.Ny / 2 + 1 + v2::z_kt(g.lNz, p->esz) - 1) / v2::z_kt(g.lNz, p->esz);
        p->cf.gx = gv; p->cd.gx = gv;
        p->ny_loc = ny; p->nq_loc = gv.hq;
        if (sharded) {
            // rows of M / H (tiles of the x kernels: 2 RP rows) and frequency pairs of this rank
            demag_status s1 = demag_shard_range(ny, world, rank, 2 * v2::x_rp(g.lLc, p->esz), &p->y0, &p->ny_loc);
            demag_status s2 = s1 ? s1 : demag_shard_range(gv.hq, world, rank, 1, &p->q0, &p->nq_loc);
            if (s2) { delete p; return s2; }
            p->cf.gx.ny = p->cd.gx.ny = p->ny_loc;
            gv.hq = p->nq_loc;                              // the y / z stages see only this rank's pairs
            p->cf.sharded = p->cd.sharded = true;
        }
        if (p->embed && !sharded && p->on[0] % 2 == 0 && !getenv("DEMAG_NO_EMBED_FUSE")) {
            p->embed_fused = true;                          // zeros supplied on load, crop on store (kernels_v2.cuh GeoV::onx)
            p->cf.gx.onx = p->cd.gx.onx = p->on[0]; p->cf.gx.ony = p->cd.gx.ony = p->on[1]; p->cf.gx.onz = p->cd.gx.onz = p->on[2];
        }
        if (sharded) p->cf.gx.ony = p->cd.gx.ony = p->ny_loc;
        p->cf.g = gv; p->cd.g = gv;
        {   // one-cell-thick mesh: y FFT . multiply . y IFFT fused in one kernel, in place on W1 (scope row a3')
            const bool film = v2::film_supported(nz, g.Nz, g.lNy, p->esz, kMaxSmem) && !getenv("DEMAG_NO_FILM");
            v2::GeoV gf = gv;
            gf.nz = ny; gf.Nz = g.Ny; gf.Ny = 1; gf.kpz = g.kpy; gf.kst = 1;
            p->cf.film = p->cd.film = film; p->cf.gfilm = p->cd.gfilm = gf;
        }
        p->cf.lLc = p->cd.lLc = g.lLc; p->cf.lNy = p->cd.lNy = g.lNy; p->cf.lNz = p->cd.lNz = g.lNz;
        p->cf.sm_count = p->cd.sm_count = p->sm_count;
        p->cf.ylong = p->cd.ylong = getenv("DEMAG_NO_YLONG") == nullptr;
        p->cf.z16 = precision == DEMAG_FP32 && getenv("DEMAG_NO_Z16") == nullptr ? (getenv("DEMAG_Z16_MINB3") ? 1 : 2) : 0;   // 2 blocks x 255 registers measured 3 % faster than 3 x 168
        p->cf.zeo = precision == DEMAG_FP32 && (g.lNz == 8 || g.lNz == 9) && g.Nz == 2 * nz && getenv("DEMAG_NO_ZEO") == nullptr;   // Nz = 128: measured slower (211 vs 150 us at C3: no pass saved there)
        p->cf.y32 = precision == DEMAG_FP32 && getenv("DEMAG_NO_Y32") == nullptr;
        {   // L2 prefetch of the tile that starts when the current one ends (kernels_v2.cuh pf_l2_*), in waves of
            // co-resident blocks; 0 = off
            float w = 0.5f;
            if (const char* e = getenv("DEMAG_PF")) { w = (float)atof(e); if (!(w >= 0.f && w <= 64.f)) w = 0.f; }
            p->cf.pf_waves = p->cd.pf_waves = w;
        }
        {   // programmatic dependent launch (profiles/r1_07_pdl.md).  Letting the next grid in at block END hides the
            // launch gap only (C3 365.6 -> 356.3 us, C2 92.0 -> 89.1 us, C4 unchanged); letting it in at block START
            // also makes its blocks resident early, which pays on launch-bound tiny meshes (C1 23.6 -> 16.4 us) and
            // costs on large ones (C3 382 us): mode 1 up to 2^16 cells, mode 2 above
            int pdl = (long long)nx * ny * nz <= (1LL << 16) ? 1 : 2;
            if (const char* e = getenv("DEMAG_PDL")) { const int v = atoi(e); if (v >= 0 && v <= 2) pdl = v; }   // A/B timing: 0 off, 1 next grid let in at block start, 2 at block end
            p->cf.pdl = p->cd.pdl = pdl != 0;
            const int trig = pdl == 2 ? 1 : 0;
            p->cf.g.trig = p->cd.g.trig = p->cf.gx.trig = p->cd.gx.trig = p->cf.gfilm.trig = p->cd.gfilm.trig = trig;
        }
        const size_t qsz = 4 * p->esz;                      // one quad
        const size_t per_q = (size_t)3 * g.nz * g.Ny * qsz;
        size_t slab_bytes = kSlabBytes;
        if (const char* e = getenv("DEMAG_SLAB_MB")) { const long long v = atoll(e); if (v >= 1 && v <= (1LL << 20)) slab_bytes = (size_t)v << 20; }
        long long n = (long long)(slab_bytes / per_q);
        if (n < 1) n = 1;
        if (n > gv.hq) n = gv.hq;
        p->nq_auto = p->nq_slab = (int)n;
        p->w1_bytes = (size_t)3 * gv.hq * g.nz * g.ny * qsz;
        if (sharded) p->w1out_bytes = (size_t)3 * (nx / 2 + 1) * g.nz * p->ny_loc * qsz;
        p->w2_bytes = (size_t)p->nq_auto * per_q;
        p->kpitch_v = gv.kst;
        p->k_bytes = (size_t)gv.hq * gv.kst * v2::z_kt(g.lNz, p->esz) * g.kpz * 12 * p->esz;     // y and z packed by symmetry
        if (p->cf.film) { p->w2_bytes = 256; p->k_bytes = (size_t)gv.hq * g.kpy * 12 * p->esz; }
    }
    auto alloc_all = [&]() -> demag_status {
        if (precision == DEMAG_FP32) { demag_status s = set_func_attrs<float>(); if (s) return s; }
        else { demag_status s = set_func_attrs<double>(); if (s) return s; }
        CUDA_TRY(cudaFuncSetAttribute(k_sym_axis, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
        CUDA_TRY(cudaFuncSetAttribute(k_sym_axis_packed, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
        {
            cudaError_t zerr = cudaSuccess;
            if (getenv("DEMAG_NO_ZSPEC")) p->z_spec = false; else
            p->z_spec = precision == DEMAG_FP32
                ? z_c_dispatch<float>(0, g, p->TY, 0, nullptr, 0, 0, nullptr, nullptr, 0, nullptr, &zerr)
                : z_c_dispatch<double>(0, g, p->TY, 0, nullptr, 0, 0, nullptr, nullptr, 0, nullptr, &zerr);
            CUDA_TRY(zerr);
        }
        if (p->v2) {
            const int LL[3] = {g.lLc, g.lNy, g.lNz};
            const int POL[3] = {v2::x_pol(g.lLc), p->cf.film ? v2::film_pol(g.lNy) : v2::y_pol(g.lNy, p->cf.y32), v2::z_pol(g.lNz)};
            cudaError_t verr = cudaSuccess;
            if (precision == DEMAG_FP32) {
                for (int a = 0; a < 3; ++a) {
                    if (a == 2 && p->cf.zeo)      // k_z_eo_v: tables of the HALF-length schedule (radix Nz/16, then 8) + w_Nz^z
                        CUDA_TRY(v2::build_axis_tables<float>(g.lNz - 1, 7, 0, &p->tf[a], nullptr, g.Nz, &p->cf.two));
                    else
                    CUDA_TRY(v2::build_axis_tables<float>(LL[a], POL[a], a == 0 ? nx : 0, &p->tf[a], a == 0 ? &p->cf.twpost : nullptr));
                    p->tw_bytes += p->tf[a].bytes;
                }
                p->cf.twx = p->tf[0].set; p->cf.twy = p->tf[1].set; p->cf.twz = p->tf[2].set;
                v2::x_fwd<float>(0, p->cf, nullptr, nullptr, nullptr, &verr); CUDA_TRY(verr);
                v2::x_inv<float>(0, p->cf, nullptr, nullptr, nullptr, &verr); CUDA_TRY(verr);
                if (p->embed_fused) {
                    v2::x_fwd_e<float>(0, p->cf, nullptr, nullptr, nullptr, &verr); CUDA_TRY(verr);
                    v2::x_inv_e<float>(0, p->cf, nullptr, nullptr, nullptr, &verr); CUDA_TRY(verr);
                }
                v2::y_fwd<float>(0, p->cf, nullptr, 0, 0, nullptr, nullptr, &verr); CUDA_TRY(verr);
                v2::y_inv<float>(0, p->cf, nullptr, 0, 0, nullptr, nullptr, &verr); CUDA_TRY(verr);
                v2::z_mul<float>(0, p->cf, nullptr, 0, 0, nullptr, nullptr, &verr); CUDA_TRY(verr);
                if (p->cf.film) { v2::y_film<float>(0, p->cf, nullptr, nullptr, nullptr, &verr); CUDA_TRY(verr); }
                if (sharded) {
                    v2::x_fwd_sh<float>(0, p->cf, nullptr, nullptr, &verr); CUDA_TRY(verr);
                    v2::y_inv_sh<float>(0, p->cf, nullptr, 0, 0, nullptr, &verr); CUDA_TRY(verr);
                }
            } else {
                for (int a = 0; a < 3; ++a) {
                    CUDA_TRY(v2::build_axis_tables<double>(LL[a], POL[a], a == 0 ? nx : 0, &p->td[a], a == 0 ? &p->cd.twpost : nullptr));
                    p->tw_bytes += p->td[a].bytes;
                }
                p->cd.twx = p->td[0].set; p->cd.twy = p->td[1].set; p->cd.twz = p->td[2].set;
                v2::x_fwd<double>(0, p->cd, nullptr, nullptr, nullptr, &verr); CUDA_TRY(verr);
                v2::x_inv<double>(0, p->cd, nullptr, nullptr, nullptr, &verr); CUDA_TRY(verr);
                if (p->embed_fused) {
                    v2::x_fwd_e<double>(0, p->cd, nullptr, nullptr, nullptr, &verr); CUDA_TRY(verr);
                    v2::x_inv_e<double>(0, p->cd, nullptr, nullptr, nullptr, &verr); CUDA_TRY(verr);
                }
                v2::y_fwd<double>(0, p->cd, nullptr, 0, 0, nullptr, nullptr, &verr); CUDA_TRY(verr);
                v2::y_inv<double>(0, p->cd, nullptr, 0, 0, nullptr, nullptr, &verr); CUDA_TRY(verr);
                v2::z_mul<double>(0, p->cd, nullptr, 0, 0, nullptr, nullptr, &verr); CUDA_TRY(verr);
                if (p->cd.film) { v2::y_film<double>(0, p->cd, nullptr, nullptr, nullptr, &verr); CUDA_TRY(verr); }
                if (sharded) {
                    v2::x_fwd_sh<double>(0, p->cd, nullptr, nullptr, &verr); CUDA_TRY(verr);
                    v2::y_inv_sh<double>(0, p->cd, nullptr, 0, 0, nullptr, &verr); CUDA_TRY(verr);
                }
            }
            {   // which kernels prefetch (bit 0 x R2C, 1 y forward, 2 z / film, 3 y inverse, 4 x C2R)
                // Measured (profiles/r2_01_prefetch.md): the y kernels gain 5-19 % (whole lines: one bulk request each), the
                // z kernel gains 11 % when its rows are >= 512 bytes (C4, 32 columns) and loses with 64-128 byte rows, the
                // x kernels do not gain (R2C) or lose (C2R: one request per 32-256 byte piece)
                // With a tensor map the whole strided tile is ONE request (profiles/r2_01_prefetch.md): the z kernel then gains
                // 4 % with narrow rows too (C3, C5), the x C2R kernel 5 % where its pieces are 32-64 bytes (long rows, C4)
                const bool z_wide = (size_t)v2::z_ty(g.lNz, p->esz) * 4 * p->esz >= 512, z_tmap = g.nz <= 256 && !getenv("DEMAG_NO_TMAP");
                int mask = 2 | 8 | (g.lNz >= 4 && (z_wide || z_tmap) ? 4 : 0) | (v2::x_rp(g.lLc, p->esz) <= 2 && !sharded && !getenv("DEMAG_NO_TMAP") ? 16 : 0);
                if (const char* e = getenv("DEMAG_PF_MASK")) mask = atoi(e);
                auto apply_mask = [&](auto& c) {
                    if (!(mask & 1)) c.pf_xf = 0;
                    if (!(mask & 2)) c.pf_yf = 0;
                    if (!(mask & 4)) { c.pf_z = 0; c.pf_film = 0; }
                    if (!(mask & 8)) c.pf_yi = 0;
                    if (!(mask & 16)) c.pf_xi = 0;
                };
                apply_mask(p->cf); apply_mask(p->cd);
            }
            {   // y position -> frequency map of the y schedule, for the plan-time pack
                const int ypol = v2::y_pol(g.lNy, p->cf.y32);
                const v2::Sched sc = v2::make_sched(g.lNy, ypol);
                std::vector<int> h((size_t)g.Ny);
                for (int q = 0; q < g.Ny; ++q) h[q] = v2::sched_freq_of_pos(sc, v2::y_w2_pos_to_tile_pos(g.lNy, ypol, q));
                CUDA_TRY(cudaMalloc(&p->ypos2freq, sizeof(int) * (size_t)g.Ny));
                CUDA_TRY(cudaMemcpy(p->ypos2freq, h.data(), sizeof(int) * (size_t)g.Ny, cudaMemcpyHostToDevice));
                p->tw_bytes += sizeof(int) * (size_t)g.Ny;
                // slots of the y-packed kernel spectrum (kernels_v2.cuh "Kv"): positions with ky <= Ny/2 in position
                // order; a mirrored position shares the slot of Ny - ky
                std::vector<int> slot_of_freq((size_t)g.Ny / 2 + 1, -1), sl((size_t)g.Ny);
                int ns = 0;
                for (int q = 0; q < g.Ny; ++q) if (2 * h[q] <= g.Ny) { slot_of_freq[h[q]] = ns; sl[q] = ns++; }
                for (int q = 0; q < g.Ny; ++q) if (2 * h[q] > g.Ny) sl[q] = slot_of_freq[g.Ny - h[q]] | (int)0x80000000;
                CUDA_TRY(cudaMalloc(&p->yslot, sizeof(int) * (size_t)g.Ny));
                CUDA_TRY(cudaMemcpy(p->yslot, sl.data(), sizeof(int) * (size_t)g.Ny, cudaMemcpyHostToDevice));
                p->tw_bytes += sizeof(int) * (size_t)g.Ny;
                p->cf.yslot = p->cd.yslot = p->yslot;
            }
        }
        if (p->embed && !p->embed_fused) {
            const size_t b = (size_t)3 * nx * ny * nz * p->esz;
            CUDA_TRY(cudaMalloc(&p->Mp, b));
            CUDA_TRY(cudaMalloc(&p->Hp, b));
            p->macro_bytes += 2 * b;
        }
        CUDA_TRY(cudaMalloc(&p->W1, p->w1_bytes));
        if (sharded) CUDA_TRY(cudaMalloc(&p->W1out, p->w1out_bytes));
        CUDA_TRY(cudaMalloc(&p->W2, p->w2_bytes));
        CUDA_TRY(cudaMalloc(&p->K, p->k_bytes));
        CUDA_TRY(cudaMemset(p->K, 0, p->k_bytes));
        if (p->v2 && !p->cf.film && !getenv("DEMAG_NO_TMAP")) {
            // tensor maps for the one-request tile prefetch (kernels_v2.cuh pf_l2_tensor); a failure only disables it
            const v2::GeoV& gv = p->cf.g;
            const unsigned long long q = 4 * p->esz;                                   // bytes per quad
            const int ty = v2::z_ty(g.lNz, p->esz);
            if (g.lNz >= 4 && g.nz <= 256 && ty * 4 <= 256) {                          // z kernel: box {TY quads, nz, 1, 3}
                const unsigned long long dim[4] = {(unsigned long long)g.Ny * 4, (unsigned long long)g.nz, (unsigned long long)p->nq_auto, 3};
                const unsigned long long sb[3] = {g.Ny * q, (unsigned long long)g.nz * g.Ny * q, (unsigned long long)p->nq_auto * g.nz * g.Ny * q};
                const unsigned box[4] = {(unsigned)ty * 4, (unsigned)g.nz, 1, 3};
                v2::TMap tm;
                if (v2::encode_tmap4(&tm, p->esz, p->W2, dim, sb, box)) { p->cf.tm_z = p->cd.tm_z = tm; p->cf.tm_z_nq = p->cd.tm_z_nq = p->nq_auto; }
                else if (ty * 4 * p->esz < 512) p->cf.pf_z = p->cd.pf_z = 0;          // no map: narrow rows do not prefetch
            }
            if (!sharded) {                                                             // x C2R: box {2 RP quads, 1, 256 pairs, 1}
                const int rp = v2::x_rp(g.lLc, p->esz);
                const unsigned long long dim[4] = {(unsigned long long)g.ny * 4, (unsigned long long)g.nz, (unsigned long long)gv.hq, 3};
                const unsigned long long sb[3] = {g.ny * q, (unsigned long long)g.nz * g.ny * q, (unsigned long long)gv.hq * g.nz * g.ny * q};
                const unsigned box[4] = {(unsigned)(2 * rp * 4), 1, (unsigned)std::min(gv.hq, 256), 1};
                v2::TMap tm;
                if (v2::encode_tmap4(&tm, p->esz, p->W1, dim, sb, box)) { p->cf.tm_xi = p->cd.tm_xi = tm; p->cf.tm_xi_ok = p->cd.tm_xi_ok = true; }
                else p->cf.pf_xi = p->cd.pf_xi = 0;
            }
        }
        const int N[3] = {g.Nx, g.Ny, g.Nz};
        for (int a = 0; a < 3; ++a) {
            demag_status s = precision == DEMAG_FP32 ? make_twiddles<float2>(N[a], &p->tw[a], &p->tw_bytes)
                                                     : make_twiddles<double2>(N[a], &p->tw[a], &p->tw_bytes);
            if (s) return s;
        }
        return DEMAG_OK;
    };
    st = alloc_all();
    if (st != DEMAG_OK) { demag_plan_destroy(p); return st; }
    *out = p;
    return DEMAG_OK;
}

demag_status demag_plan_destroy(demag_plan_t p)
{
    if (!p) return DEMAG_OK;
    for (void* q : p->ipc_open) if (q) cudaIpcCloseMemHandle(q);
    cudaFree(p->W1); cudaFree(p->W1out); cudaFree(p->W2); cudaFree(p->K);
    for (int a = 0; a < 3; ++a) cudaFree(p->tw[a]);
    cudaFree(p->Mc); cudaFree(p->Hc); cudaFree(p->Mp); cudaFree(p->Hp);
    for (int a = 0; a < 3; ++a) { cudaFree(p->tf[a].dev); cudaFree(p->td[a].dev); }
    cudaFree(p->ypos2freq); cudaFree(p->yslot);
    delete p;
    return DEMAG_OK;
}

size_t demag_workspace_bytes(demag_plan_t p)
{
    if (!p) return 0;
    return p->w1_bytes + p->w1out_bytes + p->w2_bytes + p->k_bytes + p->tw_bytes + p->macro_bytes;
}

demag_status demag_set_slab(demag_plan_t p, int kx_per_slab)
{
    if (!p) return fail(DEMAG_ERR_INVALID_ARG, "plan is NULL");
    if (kx_per_slab < 0) return fail(DEMAG_ERR_INVALID_ARG, "kx_per_slab < 0");
    if (p->v2) {                                // fast path: the slab unit is a (k, Lc-k) pair plane
        int n = kx_per_slab == 0 ? p->nq_auto : kx_per_slab;
        if (n > p->nq_auto) n = p->nq_auto;
        p->nq_slab = n;
        return DEMAG_OK;
    }
    int n = kx_per_slab == 0 ? p->nkx_auto : kx_per_slab;
    if (n > p->nkx_auto) n = p->nkx_auto;      // the W2 slab was sized for nkx_auto planes
    p->nkx_slab = n;
    return DEMAG_OK;
}

int demag_launches_per_apply(demag_plan_t p)
{
    if (!p) return 0;
    const bool copies = p->embed && !p->embed_fused;
    if (p->v2 && p->cf.film) return 3 + (copies ? 2 : 0);
    const int nslab = p->v2 ? (p->cf.g.hq + p->nq_slab - 1) / p->nq_slab : (p->g.hx + p->nkx_slab - 1) / p->nkx_slab;
    return 2 + 3 * nslab + (copies ? 2 : 0);
}

int demag_path(demag_plan_t p) { return p && p->v2 ? 1 : 0; }

demag_status demag_plan_dims(demag_plan_t p, int* nx, int* ny, int* nz, int* precision)
{
    g_err[0] = 0;
    if (!p) return fail(DEMAG_ERR_INVALID_ARG, "plan is NULL");
    if (nx) *nx = p->on[0];
    if (ny) *ny = p->sharded ? p->ny_loc : p->on[1];
    if (nz) *nz = p->on[2];
    if (precision) *precision = p->prec;
    return DEMAG_OK;
}

// llg.cu reports its errors through the same thread-local message
void demag_set_last_error_(const char* msg) { snprintf(g_err, sizeof(g_err), "%s", msg ? msg : ""); }

demag_status demag_set_pbc_images(demag_plan_t p, int images)
{
    g_err[0] = 0;
    if (!p) return fail(DEMAG_ERR_INVALID_ARG, "plan is NULL");
    if (images < 0 || images > 1000) return fail(DEMAG_ERR_INVALID_ARG, "images must be in 0..1000");
    p->pbc_images = images;
    return DEMAG_OK;
}

}  // extern "C"

// ================================================================================ plan-time: kernel
namespace {

// Real-space tensor table on the device, fp64 [6][nz][ny][nx] (built-in builder).
demag_status build_table_dev(demag_plan_s* p, double** T_out)
{
    const Geo& g = p->g;
    const size_t nc = (size_t)g.nx * g.ny * g.nz;
    double* T = nullptr;
    CUDA_TRY(cudaMalloc(&T, 6 * nc * sizeof(double)));
    if (p->pbc) {
        const int im = p->pbc_images;
        k_tensor_table_pbc<<<(unsigned)((nc + 127) / 128), 128>>>(g.nx, g.ny, g.nz, p->h[0], p->h[1], p->h[2],
            (p->pbc & DEMAG_PBC_X) ? im : -1, (p->pbc & DEMAG_PBC_Y) ? im : -1, (p->pbc & DEMAG_PBC_Z) ? im : -1, T);
    } else
    k_tensor_table<<<(unsigned)((nc + 127) / 128), 128>>>(g.nx, g.ny, g.nz, p->h[0], p->h[1], p->h[2], T);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) { cudaFree(T); return fail(DEMAG_ERR_CUDA, "k_tensor_table: %s", cudaGetErrorString(e)); }
    *T_out = T;
    return DEMAG_OK;
}

demag_status launch_sym_axis(const double* in, double* out, int n, int N, int par, int ni, size_t no,
                             size_t so_in, size_t se_in, size_t so_out, size_t se_out, const double2* tw)
{
    const int lN = ilog2(N);
    if ((size_t)N * sizeof(double2) > (size_t)kMaxSmem) {      // a 16384-point line: packed real transform, one line per block
        if (N == n || (size_t)(N / 2) * sizeof(double2) > (size_t)kMaxSmem)
            return fail(DEMAG_ERR_UNSUPPORTED, "kernel transform: a %d-point line does not fit in shared memory", N);
        const size_t grid = (size_t)ni * no;
        if (grid > 0x7fffffffULL) return fail(DEMAG_ERR_UNSUPPORTED, "kernel transform grid too large");
        k_sym_axis_packed<<<(unsigned)grid, 512, (N / 2) * sizeof(double2)>>>(in, out, n, lN, N / 2 + 1, par, ni, so_in, se_in, so_out, se_out, tw);
        CUDA_TRY(cudaGetLastError());
        return DEMAG_OK;
    }
    int B = std::max(1, std::min(8, 8192 / N));
    if (B > ni) B = ni;
    const long long elems = (long long)B * N;
    const int smem = (int)(((elems + 15) / 16 * 16) * sizeof(double2));
    const int thr = pick_threads(elems);
    const size_t tilesI = (size_t)(ni + B - 1) / B;
    const size_t grid = tilesI * no;
    if (grid > 0x7fffffffULL) return fail(DEMAG_ERR_UNSUPPORTED, "kernel transform grid too large");
    k_sym_axis<<<(unsigned)grid, thr, smem>>>(in, out, n, lN, N / 2 + 1, par, ni, B, so_in, se_in, so_out, se_out, tw);
    CUDA_TRY(cudaGetLastError());
    return DEMAG_OK;
}

template <typename T>
void launch_pack(const double* A, void* K, const Geo& g, int par_y, double scale)
{
    const size_t n = (size_t)g.hx * g.kpz * g.Ny;
    const unsigned grid = (unsigned)std::min<size_t>((n + 255) / 256, 1u << 20);
    k_pack_kernel<T><<<grid, 256>>>(A, (T*)K, g.hx, g.kpy, g.kpz, g.Ny, g.lNy, par_y, scale);
}

}  // namespace

extern "C" demag_status demag_set_kernel(demag_plan_t p, const double* N6_host)
{
    g_err[0] = 0;
    if (!p) return fail(DEMAG_ERR_INVALID_ARG, "plan is NULL");
    const Geo& g = p->g;
    const size_t nc = (size_t)g.nx * g.ny * g.nz;
    static const int par[6][3] = {{1, 1, 1}, {1, 1, 1}, {1, 1, 1}, {-1, -1, 1}, {-1, 1, -1}, {1, -1, -1}};
    double *Tdev = nullptr, *A = nullptr, *B1 = nullptr, *B2 = nullptr, *B3 = nullptr;
    double2* tw64[3] = {nullptr, nullptr, nullptr};
    size_t dummy = 0;
    demag_status st = DEMAG_OK;
    auto body = [&]() -> demag_status {
        if (!N6_host) { demag_status s = build_table_dev(p, &Tdev); if (s) return s; }
        else CUDA_TRY(cudaMalloc(&A, nc * sizeof(double)));
        CUDA_TRY(cudaMalloc(&B1, (size_t)g.nz * g.ny * g.hx * sizeof(double)));
        CUDA_TRY(cudaMalloc(&B2, (size_t)g.nz * g.kpy * g.hx * sizeof(double)));
        CUDA_TRY(cudaMalloc(&B3, (size_t)g.kpz * g.kpy * g.hx * sizeof(double)));
        const int N[3] = {g.Nx, g.Ny, g.Nz};
        for (int a = 0; a < 3; ++a) { demag_status s = make_twiddles<double2>(N[a], (void**)&tw64[a], &dummy); if (s) return s; }
        for (int c = 0; c < 6; ++c) {
            const double* src;
            if (N6_host && !p->embed) { CUDA_TRY(cudaMemcpy(A, N6_host + c * nc, nc * sizeof(double), cudaMemcpyHostToDevice)); src = A; }
            else if (N6_host) {   // caller's table covers offsets 0 <= d_a < on[a]; larger offsets never meet a cell: zero
                const size_t onc = (size_t)p->on[0] * p->on[1] * p->on[2];
                CUDA_TRY(cudaMemset(A, 0, nc * sizeof(double)));
                cudaMemcpy3DParms cp = {};
                cp.srcPtr = make_cudaPitchedPtr((void*)(N6_host + c * onc), p->on[0] * sizeof(double), p->on[0], p->on[1]);
                cp.dstPtr = make_cudaPitchedPtr(A, g.nx * sizeof(double), g.nx, g.ny);
                cp.extent = make_cudaExtent(p->on[0] * sizeof(double), p->on[1], p->on[2]);
                cp.kind = cudaMemcpyHostToDevice;
                CUDA_TRY(cudaMemcpy3D(&cp));
                src = A;
            }
            else src = Tdev + c * nc;
            demag_status s;
            // x: rows (z,y); y: lines (z; kx); z: lines (ky,kx)
            s = launch_sym_axis(src, B1, g.nx, g.Nx, par[c][0], 1, (size_t)g.nz * g.ny, g.nx, 1, g.hx, 1, tw64[0]);
            if (s) return s;
            s = launch_sym_axis(B1, B2, g.ny, g.Ny, par[c][1], g.hx, g.nz, (size_t)g.ny * g.hx, g.hx,
                                (size_t)g.kpy * g.hx, g.hx, tw64[1]);
            if (s) return s;
            s = launch_sym_axis(B2, B3, g.nz, g.Nz, par[c][2], g.kpy * g.hx, 1, 0, (size_t)g.kpy * g.hx, 0,
                                (size_t)g.kpy * g.hx, tw64[2]);
            if (s) return s;
            int nodd = 0;
            for (int a = 0; a < 3; ++a) nodd += par[c][a] < 0;
            // each odd axis contributes a factor i (X = i Im X): two odd axes -> -1.  Eq. (1)'s minus sign and
            // the inverse-transform normalisation 1/(Nx Ny Nz) are folded in here (R3).
            const double scale = (nodd == 2 ? -1.0 : 1.0) * (-1.0) / ((double)g.Nx * g.Ny * g.Nz);
            if (p->v2 && p->cf.film) {
                const v2::GeoV& gv = p->cf.g;
                const size_t n = (size_t)gv.hq * g.kpy;
                const unsigned grid = (unsigned)std::min<size_t>((n + 255) / 256, 1u << 20);
                if (p->prec == DEMAG_FP32) v2::k_pack_film_v<float><<<grid, 256>>>(B3, (float*)p->K, c, gv.Lc, gv.hq, g.kpy, 0.5 * scale);
                else v2::k_pack_film_v<double><<<grid, 256>>>(B3, (double*)p->K, c, gv.Lc, gv.hq, g.kpy, 0.5 * scale);
            }
            else if (p->v2) {    // pair layout; the real split of the x transform hands over 2 X[k]: fold the 1/2 here
                const v2::GeoV& gv = p->cf.g;
                const size_t n = (size_t)gv.hq * g.kpz * g.Ny;
                const unsigned grid = (unsigned)std::min<size_t>((n + 255) / 256, 1u << 20);
                if (p->prec == DEMAG_FP32)
                    v2::k_pack_kernel_v<float><<<grid, 256>>>(B3, (float*)p->K, c, gv.Lc, gv.hq, g.kpy, g.kpz, g.Ny, v2::z_kt(g.lNz, p->esz), p->kpitch_v, p->ypos2freq, p->yslot, 0.5 * scale, p->q0);
                else
                    v2::k_pack_kernel_v<double><<<grid, 256>>>(B3, (double*)p->K, c, gv.Lc, gv.hq, g.kpy, g.kpz, g.Ny, v2::z_kt(g.lNz, p->esz), p->kpitch_v, p->ypos2freq, p->yslot, 0.5 * scale, p->q0);
            }
            else if (p->prec == DEMAG_FP32) launch_pack<float>(B3, (char*)p->K + c * p->kcomp_stride * p->esz, g, par[c][1], scale);
            else launch_pack<double>(B3, (char*)p->K + c * p->kcomp_stride * p->esz, g, par[c][1], scale);
            CUDA_TRY(cudaGetLastError());
        }
        CUDA_TRY(cudaDeviceSynchronize());
        return DEMAG_OK;
    };
    st = body();
    cudaFree(Tdev); cudaFree(A); cudaFree(B1); cudaFree(B2); cudaFree(B3);
    for (int a = 0; a < 3; ++a) cudaFree(tw64[a]);
    if (st == DEMAG_OK) p->has_kernel = true;
    return st;
}

extern "C" demag_status demag_get_kernel_real(demag_plan_t p, double* N6_host)
{
    g_err[0] = 0;
    if (!p || !N6_host) return fail(DEMAG_ERR_INVALID_ARG, "NULL argument");
    double* T = nullptr;
    demag_status st = build_table_dev(p, &T);
    if (st) return st;
    const size_t nc = (size_t)p->g.nx * p->g.ny * p->g.nz;
    cudaError_t e = cudaSuccess;
    if (!p->embed) e = cudaMemcpy(N6_host, T, 6 * nc * sizeof(double), cudaMemcpyDeviceToHost);
    else {
        const size_t onc = (size_t)p->on[0] * p->on[1] * p->on[2];
        for (int c = 0; c < 6 && e == cudaSuccess; ++c) {
            cudaMemcpy3DParms cp = {};
            cp.srcPtr = make_cudaPitchedPtr(T + c * nc, p->g.nx * sizeof(double), p->g.nx, p->g.ny);
            cp.dstPtr = make_cudaPitchedPtr(N6_host + c * onc, p->on[0] * sizeof(double), p->on[0], p->on[1]);
            cp.extent = make_cudaExtent(p->on[0] * sizeof(double), p->on[1], p->on[2]);
            cp.kind = cudaMemcpyDeviceToHost;
            e = cudaMemcpy3D(&cp);
        }
    }
    cudaFree(T);
    if (e != cudaSuccess) return fail(DEMAG_ERR_CUDA, "copy back: %s", cudaGetErrorString(e));
    return DEMAG_OK;
}

// ================================================================================ hot path
namespace {

// Optional per-launch event recorder used only by demag_apply_profiled.
struct StageTimer {
    std::vector<cudaEvent_t> ev;   // pairs
    std::vector<int> stage;
    cudaStream_t st;
    void begin(int s) { cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b); cudaEventRecord(a, st); ev.push_back(a); ev.push_back(b); stage.push_back(s); }
    void end() { cudaEventRecord(ev.back(), st); }
};
#define STAGE(s, launch) do { if (tm) tm->begin(s); launch; if (tm) tm->end(); } while (0)

template <typename T> const v2::Ctx<T>& v2_ctx(const demag_plan_s* p);
template <> const v2::Ctx<float>& v2_ctx<float>(const demag_plan_s* p) { return p->cf; }
template <> const v2::Ctx<double>& v2_ctx<double>(const demag_plan_s* p) { return p->cd; }

template <typename T>
demag_status apply_impl(demag_plan_s* p, const T* M, T* H, cudaStream_t st, StageTimer* tm = nullptr, int acc = 0)
{
    using C = typename cx_of<T>::type;
    const Geo& g = p->g;
    Geo ga = g; ga.acc = acc;                       // the x C2R kernels add into H when asked (demag_apply_add)
    C* W1 = (C*)p->W1; C* W2 = (C*)p->W2;
    const C* twx = (const C*)p->tw[0]; const C* twy = (const C*)p->tw[1]; const C* twz = (const C*)p->tw[2];
    const size_t nc = (size_t)g.nx * g.ny * g.nz;
    if (p->v2) {
        const v2::Ctx<T>& cx = v2_ctx<T>(p);
        v2::CQ<T>* V1 = (v2::CQ<T>*)p->W1; v2::CQ<T>* V2 = (v2::CQ<T>*)p->W2;
        const typename v2::kchunks<T>::V* Kv = (const typename v2::kchunks<T>::V*)p->K;
        cudaError_t verr = cudaSuccess;
        bool ok = true;             // a launcher returns false when no kernel is instantiated for the size (a stage would be skipped)
        if (p->embed_fused) STAGE(0, (ok &= v2::x_fwd_e<T>(1, cx, st, M, V1, &verr)));
        else STAGE(0, (ok &= v2::x_fwd<T>(1, cx, st, M, V1, &verr)));
        if (cx.film) STAGE(2, (ok &= v2::y_film<T>(1, cx, st, V1, Kv, &verr)));
        else for (int q0 = 0; q0 < cx.g.hq; q0 += p->nq_slab) {
            const int nq = std::min(p->nq_slab, cx.g.hq - q0);
            STAGE(1, (ok &= v2::y_fwd<T>(1, cx, st, q0, nq, V1, V2, &verr)));
            STAGE(2, (ok &= v2::z_mul<T>(1, cx, st, q0, nq, V2, Kv, &verr)));
            STAGE(3, (ok &= v2::y_inv<T>(1, cx, st, q0, nq, V2, V1, &verr)));
        }
        if (p->embed_fused) STAGE(4, (ok &= v2::x_inv_e<T>(1, cx, st, V1, H, &verr, acc)));
        else STAGE(4, (ok &= v2::x_inv<T>(1, cx, st, V1, H, &verr, acc)));
        if (!ok) return fail(DEMAG_ERR_UNSUPPORTED, "no kernel instantiated for a stage of this plan (fast family)");
        CUDA_TRY(cudaGetLastError());
        return DEMAG_OK;
    }
    if (g.Nx == 1) {
        const unsigned grid = (unsigned)std::min<size_t>((3 * nc + 255) / 256, (size_t)p->sm_count * 16);
        STAGE(0, (k_x_copy_fwd<T><<<grid, 256, 0, st>>>(3 * nc, M, W1)));
    } else {
        if (p->fast1) STAGE(0, (k_x_r2c_f<T><<<3u * g.nz * (g.ny / p->R1), p->thr1, p->smem1, st>>>(g, p->R1, p->pitch1, M, W1, twx)));
        else if (p->pitch1 == 1) STAGE(0, (k_x_r2c<T, true><<<3u * g.nz * (g.ny / p->R1), p->thr1, p->smem1, st>>>(g, p->R1, p->pitch1, M, W1, twx)));
        else STAGE(0, (k_x_r2c<T, false><<<3u * g.nz * (g.ny / p->R1), p->thr1, p->smem1, st>>>(g, p->R1, p->pitch1, M, W1, twx)));
    }
    for (int kx0 = 0; kx0 < g.hx; kx0 += p->nkx_slab) {
        const int nkx = std::min(p->nkx_slab, g.hx - kx0);
        const unsigned g2 = (unsigned)((3LL * nkx * g.nz + p->B2 - 1) / p->B2);
        if (p->fast2) STAGE(1, (k_y_fwd_f<T><<<g2, p->thr2, p->smem2, st>>>(g, p->B2, p->pitch2, kx0, nkx, W1, W2, twy)));
        else if (p->pitch2 == 1) STAGE(1, (k_y_fwd<T, true><<<g2, p->thr2, p->smem2, st>>>(g, p->B2, p->pitch2, kx0, nkx, W1, W2, twy)));
        else STAGE(1, (k_y_fwd<T, false><<<g2, p->thr2, p->smem2, st>>>(g, p->B2, p->pitch2, kx0, nkx, W1, W2, twy)));
        const unsigned g3 = (unsigned)(nkx * (g.Ny / p->TY));
        const T* Kp = (const T*)p->K;
        cudaError_t zerr = cudaSuccess;
        if (p->z_spec) STAGE(2, (z_c_dispatch<T>(1, g, p->TY, g3, st, kx0, nkx, W2, Kp, p->kcomp_stride, twz, &zerr)));
        else if (g.lNz <= 3) STAGE(2, (k_z_small<T><<<g3, p->thr3, 0, st>>>(g, p->TY, kx0, nkx, W2, Kp, p->kcomp_stride)));
        else if (g.lNz % 3 == 1) STAGE(2, (k_z_mul<T, 1><<<g3, p->thr3, p->smem3, st>>>(g, p->TY, kx0, nkx, W2, Kp, p->kcomp_stride, twz)));
        else if (g.lNz % 3 == 2) STAGE(2, (k_z_mul<T, 2><<<g3, p->thr3, p->smem3, st>>>(g, p->TY, kx0, nkx, W2, Kp, p->kcomp_stride, twz)));
        else STAGE(2, (k_z_mul<T, 3><<<g3, p->thr3, p->smem3, st>>>(g, p->TY, kx0, nkx, W2, Kp, p->kcomp_stride, twz)));
        if (p->fast2) STAGE(3, (k_y_inv_f<T><<<g2, p->thr2, p->smem2, st>>>(g, p->B2, p->pitch2, kx0, nkx, W2, W1, twy)));
        else if (p->pitch2 == 1) STAGE(3, (k_y_inv<T, true><<<g2, p->thr2, p->smem2, st>>>(g, p->B2, p->pitch2, kx0, nkx, W2, W1, twy)));
        else STAGE(3, (k_y_inv<T, false><<<g2, p->thr2, p->smem2, st>>>(g, p->B2, p->pitch2, kx0, nkx, W2, W1, twy)));
    }
    if (g.Nx == 1) {
        const unsigned grid = (unsigned)std::min<size_t>((3 * nc + 255) / 256, (size_t)p->sm_count * 16);
        STAGE(4, (k_x_copy_inv<T><<<grid, 256, 0, st>>>(3 * nc, W1, H, acc)));
    } else {
        if (p->fast1) STAGE(4, (k_x_c2r_f<T><<<3u * g.nz * (g.ny / p->R1), p->thr1, p->smem1, st>>>(ga, p->R1, p->pitch1, W1, H, twx)));
        else if (p->pitch1 == 1) STAGE(4, (k_x_c2r<T, true><<<3u * g.nz * (g.ny / p->R1), p->thr1, p->smem1, st>>>(ga, p->R1, p->pitch1, W1, H, twx)));
        else STAGE(4, (k_x_c2r<T, false><<<3u * g.nz * (g.ny / p->R1), p->thr1, p->smem1, st>>>(ga, p->R1, p->pitch1, W1, H, twx)));
    }
    CUDA_TRY(cudaGetLastError());
    return DEMAG_OK;
}

// caller's mesh <-> embedding power-of-two mesh (only for plans with embed == true)
template <typename T>
__global__ void __launch_bounds__(256) k_embed(int onx, int ony, int onz, int nx, int ny, int nz, const T* __restrict__ M, T* __restrict__ Mp)
{
    const int y = blockIdx.y, cz = blockIdx.z, c = cz / nz, z = cz - c * nz;
    const bool in = y < ony && z < onz;
    const T* src = M + (((size_t)c * onz + z) * ony + y) * onx;
    T* dst = Mp + (((size_t)c * nz + z) * ny + y) * nx;
    for (int x = blockIdx.x * 256 + threadIdx.x; x < nx; x += gridDim.x * 256) dst[x] = (in && x < onx) ? src[x] : (T)0;
}
template <typename T>
__global__ void __launch_bounds__(256) k_crop(int onx, int ony, int onz, int nx, int ny, int nz, const T* __restrict__ Hp, T* __restrict__ H, int acc)
{
    const int y = blockIdx.y, cz = blockIdx.z, c = cz / onz, z = cz - c * onz;
    const T* src = Hp + (((size_t)c * nz + z) * ny + y) * nx;
    T* dst = H + (((size_t)c * onz + z) * ony + y) * onx;
    for (int x = blockIdx.x * 256 + threadIdx.x; x < onx; x += gridDim.x * 256) dst[x] = acc ? dst[x] + src[x] : src[x];
}
// demag_apply on the caller's mesh
template <typename T>
demag_status apply_outer(demag_plan_s* p, const T* M, T* H, cudaStream_t st, StageTimer* tm = nullptr, int acc = 0)
{
    if (!p->embed || p->embed_fused) return apply_impl<T>(p, M, H, st, tm, acc);
    const Geo& g = p->g;
    k_embed<T><<<dim3((unsigned)((g.nx + 255) / 256), (unsigned)g.ny, (unsigned)(3 * g.nz)), 256, 0, st>>>(
        p->on[0], p->on[1], p->on[2], g.nx, g.ny, g.nz, M, (T*)p->Mp);
    demag_status s = apply_impl<T>(p, (const T*)p->Mp, (T*)p->Hp, st, tm);
    if (s) return s;
    k_crop<T><<<dim3((unsigned)((p->on[0] + 255) / 256), (unsigned)p->on[1], (unsigned)(3 * p->on[2])), 256, 0, st>>>(
        p->on[0], p->on[1], p->on[2], g.nx, g.ny, g.nz, (const T*)p->Hp, H, acc);
    CUDA_TRY(cudaGetLastError());
    return DEMAG_OK;
}

demag_status check_apply_args(demag_plan_s* p, const void* a, const void* b, size_t bytes)
{
    if (!p) return fail(DEMAG_ERR_INVALID_ARG, "plan is NULL");
    if (p->sharded && p->world > 1) return fail(DEMAG_ERR_INVALID_ARG, "plan is one rank of %d: use demag_apply_sharded", p->world);
    if (!a || !b) return fail(DEMAG_ERR_INVALID_ARG, "NULL device pointer");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device)
        return fail(DEMAG_ERR_INVALID_ARG, "plan was created on device %d, the current device is %d", p->device, dev);
    if (((uintptr_t)a & 15) || ((uintptr_t)b & 15)) return fail(DEMAG_ERR_INVALID_ARG, "device pointers must be 16-byte aligned");
    const char *pa = (const char*)a, *pb = (const char*)b;
    if (pa < pb + bytes && pb < pa + bytes) return fail(DEMAG_ERR_INVALID_ARG, "input and output overlap");
    return DEMAG_OK;
}

}  // namespace

extern "C" demag_status demag_apply(demag_plan_t p, const void* M_dev, void* H_dev, void* cuda_stream)
{
    g_err[0] = 0;
    if (!p) return fail(DEMAG_ERR_INVALID_ARG, "plan is NULL");
    const size_t bytes = (size_t)3 * p->on[0] * p->on[1] * p->on[2] * p->esz;
    demag_status s = check_apply_args(p, M_dev, H_dev, bytes);
    if (s) return s;
    if (!p->has_kernel) return fail(DEMAG_ERR_NO_KERNEL, "demag_set_kernel has not been called");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    return p->prec == DEMAG_FP32 ? apply_outer<float>(p, (const float*)M_dev, (float*)H_dev, st)
                                 : apply_outer<double>(p, (const double*)M_dev, (double*)H_dev, st);
}

extern "C" demag_status demag_apply_add(demag_plan_t p, const void* M_dev, void* Heff_dev, void* cuda_stream)
{
    g_err[0] = 0;
    if (!p) return fail(DEMAG_ERR_INVALID_ARG, "plan is NULL");
    const size_t bytes = (size_t)3 * p->on[0] * p->on[1] * p->on[2] * p->esz;
    demag_status s = check_apply_args(p, M_dev, Heff_dev, bytes);
    if (s) return s;
    if (!p->has_kernel) return fail(DEMAG_ERR_NO_KERNEL, "demag_set_kernel has not been called");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    return p->prec == DEMAG_FP32 ? apply_outer<float>(p, (const float*)M_dev, (float*)Heff_dev, st, nullptr, 1)
                                 : apply_outer<double>(p, (const double*)M_dev, (double*)Heff_dev, st, nullptr, 1);
}

// ================================================================================ several GPUs
extern "C" demag_status demag_shard_info(demag_plan_t p, int* rank, int* world, int* y0, int* ny_loc, int* q0, int* nq_loc)
{
    g_err[0] = 0;
    if (!p) return fail(DEMAG_ERR_INVALID_ARG, "plan is NULL");
    if (!p->sharded) return fail(DEMAG_ERR_INVALID_ARG, "plan was not created by demag_plan_create_sharded");
    if (rank) *rank = p->rank;
    if (world) *world = p->world;
    if (y0) *y0 = p->y0;
    if (ny_loc) *ny_loc = p->ny_loc;
    if (q0) *q0 = p->q0;
    if (nq_loc) *nq_loc = p->nq_loc;
    return DEMAG_OK;
}

extern "C" demag_status demag_shard_buffers(demag_plan_t p, void** w1in_dev, size_t* w1in_bytes, void** w1out_dev, size_t* w1out_bytes)
{
    g_err[0] = 0;
    if (!p) return fail(DEMAG_ERR_INVALID_ARG, "plan is NULL");
    if (!p->sharded) return fail(DEMAG_ERR_INVALID_ARG, "plan was not created by demag_plan_create_sharded");
    if (w1in_dev) *w1in_dev = p->W1;
    if (w1in_bytes) *w1in_bytes = p->w1_bytes;
    if (w1out_dev) *w1out_dev = p->W1out;
    if (w1out_bytes) *w1out_bytes = p->w1out_bytes;
    return DEMAG_OK;
}

namespace {
template <typename T>
void install_peers(demag_plan_s* p, v2::Ctx<T>& c, void* const* in, void* const* outp)
{
    const int hq = p->g.nx / 2 + 1;
    int b0 = 0, cnt = 0;
    // x R2C -> W1in of the pair's owner: pairs per rank, this rank's first row, row length = whole ny
    demag_shard_range(hq, p->world, 0, 1, &b0, &cnt);
    c.m_in.G = p->world; c.m_in.per = cnt; c.m_in.total = hq; c.m_in.off = p->y0; c.m_in.pitch = p->g.ny;
    // y inverse -> W1out of the row's owner: rows per rank, this rank's first pair, pairs = whole hq
    demag_shard_range(p->g.ny, p->world, 0, 2 * v2::x_rp(p->g.lLc, p->esz), &b0, &cnt);
    c.m_out.G = p->world; c.m_out.per = cnt; c.m_out.total = p->g.ny; c.m_out.off = p->q0; c.m_out.pitch = hq;
    for (int r = 0; r < v2::kMaxRanks; ++r) {
        c.m_in.base[r] = r < p->world ? (v2::CQ<T>*)in[r] : nullptr;
        c.m_out.base[r] = r < p->world ? (v2::CQ<T>*)outp[r] : nullptr;
    }
}
}  // namespace

extern "C" demag_status demag_shard_set_peers(demag_plan_t p, void* const* w1in_of_rank, void* const* w1out_of_rank)
{
    g_err[0] = 0;
    if (!p || !w1in_of_rank || !w1out_of_rank) return fail(DEMAG_ERR_INVALID_ARG, "NULL argument");
    if (!p->sharded) return fail(DEMAG_ERR_INVALID_ARG, "plan was not created by demag_plan_create_sharded");
    for (int r = 0; r < p->world; ++r)
        if (!w1in_of_rank[r] || !w1out_of_rank[r] || ((uintptr_t)w1in_of_rank[r] & 15) || ((uintptr_t)w1out_of_rank[r] & 15))
            return fail(DEMAG_ERR_INVALID_ARG, "buffer of rank %d is NULL or not 16-byte aligned", r);
    if (w1in_of_rank[p->rank] != p->W1 || w1out_of_rank[p->rank] != p->W1out)
        return fail(DEMAG_ERR_INVALID_ARG, "entry %d must be this plan's own buffers (demag_shard_buffers)", p->rank);
    if (p->prec == DEMAG_FP32) install_peers<float>(p, p->cf, w1in_of_rank, w1out_of_rank);
    else install_peers<double>(p, p->cd, w1in_of_rank, w1out_of_rank);
    p->peers_set = true;
    return DEMAG_OK;
}

extern "C" demag_status demag_shard_ipc_export(demag_plan_t p, void* handles_host)
{
    g_err[0] = 0;
    if (!p || !handles_host) return fail(DEMAG_ERR_INVALID_ARG, "NULL argument");
    if (!p->sharded) return fail(DEMAG_ERR_INVALID_ARG, "plan was not created by demag_plan_create_sharded");
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "two 64-byte handles per rank");
    cudaIpcMemHandle_t h[2];
    CUDA_TRY(cudaIpcGetMemHandle(&h[0], p->W1));
    CUDA_TRY(cudaIpcGetMemHandle(&h[1], p->W1out));
    memcpy(handles_host, h, sizeof(h));
    return DEMAG_OK;
}

extern "C" demag_status demag_shard_ipc_connect(demag_plan_t p, const void* all_handles_host)
{
    g_err[0] = 0;
    if (!p || !all_handles_host) return fail(DEMAG_ERR_INVALID_ARG, "NULL argument");
    if (!p->sharded) return fail(DEMAG_ERR_INVALID_ARG, "plan was not created by demag_plan_create_sharded");
    if (p->peers_set) return fail(DEMAG_ERR_INVALID_ARG, "peers are already installed");
    void* in[v2::kMaxRanks]; void* outp[v2::kMaxRanks];
    for (int r = 0; r < p->world; ++r) {
        if (r == p->rank) { in[r] = p->W1; outp[r] = p->W1out; continue; }
        cudaIpcMemHandle_t h[2];
        memcpy(h, (const char*)all_handles_host + (size_t)r * sizeof(h), sizeof(h));
        CUDA_TRY(cudaIpcOpenMemHandle(&p->ipc_open[2 * r], h[0], cudaIpcMemLazyEnablePeerAccess));
        CUDA_TRY(cudaIpcOpenMemHandle(&p->ipc_open[2 * r + 1], h[1], cudaIpcMemLazyEnablePeerAccess));
        in[r] = p->ipc_open[2 * r]; outp[r] = p->ipc_open[2 * r + 1];
    }
    return demag_shard_set_peers(p, in, outp);
}

namespace {
template <typename T>
demag_status apply_sharded_impl(demag_plan_s* p, int phase, const T* M, T* H, cudaStream_t st)
{
    const v2::Ctx<T>& cx = v2_ctx<T>(p);
    cudaError_t verr = cudaSuccess;
    if (phase == 0) v2::x_fwd_sh<T>(1, cx, st, M, &verr);                         // xFFT_R2C + Transfer_S1_to_S2
    else if (phase == 1) {
        v2::CQ<T>* V1 = (v2::CQ<T>*)p->W1; v2::CQ<T>* V2 = (v2::CQ<T>*)p->W2;
        const typename v2::kchunks<T>::V* Kv = (const typename v2::kchunks<T>::V*)p->K;
        for (int q0 = 0; q0 < cx.g.hq; q0 += p->nq_slab) {                        // this rank's pairs, slab by slab
            const int nq = std::min(p->nq_slab, cx.g.hq - q0);
            v2::y_fwd<T>(1, cx, st, q0, nq, V1, V2, &verr);
            v2::z_mul<T>(1, cx, st, q0, nq, V2, Kv, &verr);
            v2::y_inv_sh<T>(1, cx, st, q0, nq, V2, &verr);                        // yFFT inverse + Transfer_S2_to_S1
        }
    }
    else v2::x_inv<T>(1, cx, st, (const v2::CQ<T>*)p->W1out, H, &verr, 0);        // xFFT_C2R
    CUDA_TRY(cudaGetLastError());
    return DEMAG_OK;
}
}  // namespace

extern "C" demag_status demag_apply_sharded(demag_plan_t p, int phase, const void* M_loc_dev, void* H_loc_dev, void* cuda_stream)
{
    g_err[0] = 0;
    if (!p) return fail(DEMAG_ERR_INVALID_ARG, "plan is NULL");
    if (!p->sharded) return fail(DEMAG_ERR_INVALID_ARG, "plan was not created by demag_plan_create_sharded");
    if (phase < 0 || phase > 2) return fail(DEMAG_ERR_INVALID_ARG, "phase must be 0, 1 or 2");
    if (!p->peers_set) return fail(DEMAG_ERR_INVALID_ARG, "peers not installed (demag_shard_ipc_connect / demag_shard_set_peers)");
    if (!p->has_kernel) return fail(DEMAG_ERR_NO_KERNEL, "demag_set_kernel has not been called");
    const void* io = phase == 0 ? M_loc_dev : phase == 2 ? H_loc_dev : (const void*)p->W1;
    if (!io) return fail(DEMAG_ERR_INVALID_ARG, "NULL device pointer");
    if ((uintptr_t)io & 15) return fail(DEMAG_ERR_INVALID_ARG, "device pointers must be 16-byte aligned");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    return p->prec == DEMAG_FP32 ? apply_sharded_impl<float>(p, phase, (const float*)M_loc_dev, (float*)H_loc_dev, st)
                                 : apply_sharded_impl<double>(p, phase, (const double*)M_loc_dev, (double*)H_loc_dev, st);
}

extern "C" demag_status demag_apply_profiled(demag_plan_t p, const void* M_dev, void* H_dev, void* cuda_stream,
                                             float* stage_ms_host, int* stage_launches_host)
{
    g_err[0] = 0;
    if (!p) return fail(DEMAG_ERR_INVALID_ARG, "plan is NULL");
    const size_t bytes = (size_t)3 * p->on[0] * p->on[1] * p->on[2] * p->esz;
    demag_status s = check_apply_args(p, M_dev, H_dev, bytes);
    if (s) return s;
    if (!p->has_kernel) return fail(DEMAG_ERR_NO_KERNEL, "demag_set_kernel has not been called");
    StageTimer tm;
    tm.st = (cudaStream_t)cuda_stream;
    s = p->prec == DEMAG_FP32 ? apply_outer<float>(p, (const float*)M_dev, (float*)H_dev, tm.st, &tm)
                              : apply_outer<double>(p, (const double*)M_dev, (double*)H_dev, tm.st, &tm);
    cudaError_t e = cudaStreamSynchronize(tm.st);
    float ms[5] = {0, 0, 0, 0, 0};
    int cnt[5] = {0, 0, 0, 0, 0};
    for (size_t i = 0; i < tm.stage.size(); ++i) {
        float t = 0.f;
        if (e == cudaSuccess) cudaEventElapsedTime(&t, tm.ev[2 * i], tm.ev[2 * i + 1]);
        ms[tm.stage[i]] += t; cnt[tm.stage[i]]++;
        cudaEventDestroy(tm.ev[2 * i]); cudaEventDestroy(tm.ev[2 * i + 1]);
    }
    if (stage_ms_host) memcpy(stage_ms_host, ms, sizeof(ms));
    if (stage_launches_host) memcpy(stage_launches_host, cnt, sizeof(cnt));
    if (s) return s;
    if (e != cudaSuccess) return fail(DEMAG_ERR_CUDA, "profiled apply: %s", cudaGetErrorString(e));
    return DEMAG_OK;
}

extern "C" demag_status demag_energy(demag_plan_t p, const void* M_dev, const void* H_dev, double* E_dev, void* cuda_stream)
{
    g_err[0] = 0;
    if (!p || !M_dev || !H_dev || !E_dev) return fail(DEMAG_ERR_INVALID_ARG, "NULL argument");
    if ((uintptr_t)E_dev & 7) return fail(DEMAG_ERR_INVALID_ARG, "E_dev must be 8-byte aligned");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n3 = (size_t)3 * p->on[0] * (p->sharded ? p->ny_loc : p->on[1]) * p->on[2];   // sharded: this rank's rows
    const double mu0 = 4.0e-7 * 3.14159265358979323846;
    const double scale = -0.5 * mu0 * p->h[0] * p->h[1] * p->h[2];
    CUDA_TRY(cudaMemsetAsync(E_dev, 0, sizeof(double), st));
    const unsigned grid = (unsigned)std::min<size_t>((n3 + 255) / 256, (size_t)p->sm_count * 8);
    if (p->prec == DEMAG_FP32) k_energy<float><<<grid, 256, 0, st>>>(n3, (const float*)M_dev, (const float*)H_dev, scale, E_dev);
    else k_energy<double><<<grid, 256, 0, st>>>(n3, (const double*)M_dev, (const double*)H_dev, scale, E_dev);
    CUDA_TRY(cudaGetLastError());
    return DEMAG_OK;
}

namespace {
template <typename T>
demag_status extrapolate_impl(demag_plan_s* p, int npts, const void* const* H, const double* w, void* out, int acc,
                              size_t n, cudaStream_t st)
{
    ExtrapArgs<T> a;
    for (int k = 0; k < kMaxHist; ++k) { a.H[k] = k < npts ? (const T*)H[k] : nullptr; a.w[k] = k < npts ? (T)w[k] : (T)0; }
    const unsigned grid = (unsigned)std::min<size_t>((n / (16 / sizeof(T)) + 255) / 256 + 1, (size_t)p->sm_count * 8);
    switch (npts) {
#define DEMAG_EXTRAP_CASE(NP) case NP: k_extrapolate<T, NP><<<grid, 256, 0, st>>>(n, a, (T*)out, acc); break;
        DEMAG_EXTRAP_CASE(1) DEMAG_EXTRAP_CASE(2) DEMAG_EXTRAP_CASE(3) DEMAG_EXTRAP_CASE(4)
        DEMAG_EXTRAP_CASE(5) DEMAG_EXTRAP_CASE(6) DEMAG_EXTRAP_CASE(7) DEMAG_EXTRAP_CASE(8)
#undef DEMAG_EXTRAP_CASE
    }
    CUDA_TRY(cudaGetLastError());
    return DEMAG_OK;
}
}  // namespace

extern "C" demag_status demag_extrapolate(demag_plan_t p, int npts, const void* const* H_hist_dev, const double* t_hist_host,
                                          double t, void* H_out_dev, int accumulate, void* cuda_stream)
{
    g_err[0] = 0;
    if (!p || !H_hist_dev || !t_hist_host || !H_out_dev) return fail(DEMAG_ERR_INVALID_ARG, "NULL argument");
    if (npts < 1 || npts > kMaxHist) return fail(DEMAG_ERR_INVALID_ARG, "npts must be in 1..%d", kMaxHist);
    if (!isfinite(t)) return fail(DEMAG_ERR_INVALID_ARG, "t is not finite");
    const size_t n = (size_t)3 * p->on[0] * (p->sharded ? p->ny_loc : p->on[1]) * p->on[2];
    const size_t bytes = n * p->esz;
    if ((uintptr_t)H_out_dev & 15) return fail(DEMAG_ERR_INVALID_ARG, "device pointers must be 16-byte aligned");
    double w[kMaxHist];
    for (int k = 0; k < npts; ++k) {
        if (!H_hist_dev[k] || ((uintptr_t)H_hist_dev[k] & 15)) return fail(DEMAG_ERR_INVALID_ARG, "field %d is NULL or not 16-byte aligned", k);
        const char *pa = (const char*)H_hist_dev[k], *pb = (const char*)H_out_dev;
        if (pa < pb + bytes && pb < pa + bytes) return fail(DEMAG_ERR_INVALID_ARG, "field %d overlaps the output", k);
        if (!isfinite(t_hist_host[k])) return fail(DEMAG_ERR_INVALID_ARG, "time %d is not finite", k);
        long double L = 1.0L;                                  // Lagrange weight L_k(t), PAPER.md:96 / R19
        for (int j = 0; j < npts; ++j) {
            if (j == k) continue;
            if (t_hist_host[j] == t_hist_host[k]) return fail(DEMAG_ERR_INVALID_ARG, "times %d and %d coincide", j, k);
            L *= ((long double)t - t_hist_host[j]) / ((long double)t_hist_host[k] - t_hist_host[j]);
        }
        w[k] = (double)L;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    return p->prec == DEMAG_FP32 ? extrapolate_impl<float>(p, npts, H_hist_dev, w, H_out_dev, accumulate != 0, n, st)
                                 : extrapolate_impl<double>(p, npts, H_hist_dev, w, H_out_dev, accumulate != 0, n, st);
}

extern "C" demag_status demag_atomistic_reserve(demag_plan_t p)
{
    g_err[0] = 0;
    if (!p) return fail(DEMAG_ERR_INVALID_ARG, "plan is NULL");
    if (p->Mc && p->Hc) return DEMAG_OK;
    const size_t b = (size_t)3 * p->on[0] * p->on[1] * p->on[2] * p->esz;
    if (!p->Mc) CUDA_TRY(cudaMalloc(&p->Mc, b));
    if (!p->Hc) CUDA_TRY(cudaMalloc(&p->Hc, b));
    p->macro_bytes += 2 * b;
    return DEMAG_OK;
}

extern "C" demag_status demag_apply_atomistic(demag_plan_t p, const void* S_dev, void* Hs_dev, int cx, int cy, int cz,
                                              double mu_s_in_muB, double a, int accumulate, void* cuda_stream)
{
    g_err[0] = 0;
    if (!p) return fail(DEMAG_ERR_INVALID_ARG, "plan is NULL");
    if (cx < 1 || cy < 1 || cz < 1 || !(a > 0) || !isfinite(mu_s_in_muB))
        return fail(DEMAG_ERR_INVALID_ARG, "bad macrocell / lattice arguments");
    struct { int nx, ny, nz; } g = {p->on[0], p->on[1], p->on[2]};     // the caller's macrocell mesh
    const double want[3] = {cx * a, cy * a, cz * a};
    for (int i = 0; i < 3; ++i)
        if (fabs(want[i] - p->h[i]) > 1e-9 * p->h[i])
            return fail(DEMAG_ERR_INVALID_ARG, "plan cell size must equal macrocell size c*a (axis %d)", i);
    const size_t nspin3 = (size_t)3 * g.nx * cx * g.ny * cy * g.nz * cz;
    demag_status s = check_apply_args(p, S_dev, Hs_dev, nspin3 * p->esz);
    if (s) return s;
    if (!p->has_kernel) return fail(DEMAG_ERR_NO_KERNEL, "demag_set_kernel has not been called");
    const size_t nc = (size_t)g.nx * g.ny * g.nz;
    if (!p->Mc || !p->Hc) return fail(DEMAG_ERR_INVALID_ARG, "macrocell arrays not allocated: call demag_atomistic_reserve first");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const double muB = 9.2740100783e-24;
    const double f = muB * mu_s_in_muB / ((double)cx * cy * cz * a * a * a);
    const unsigned ga = (unsigned)std::min<size_t>((3 * nc + 255) / 256, (size_t)1 << 22);
    const unsigned gs = (unsigned)std::min<size_t>((nspin3 / 4 + 255) / 256 + 1, (size_t)p->sm_count * 32);
    if (p->prec == DEMAG_FP32 && cx == 4 && g.ny <= 65535 && 3 * g.nz <= 65535) {
        const dim3 g3((unsigned)((g.nx + 127) / 128), (unsigned)g.ny, (unsigned)(3 * g.nz));
        k_macro_avg_x4<<<g3, 128, 0, st>>>(g.nx, cy, cz, (const float*)S_dev, (float*)p->Mc, f);
        s = apply_outer<float>(p, (const float*)p->Mc, (float*)p->Hc, st);
        if (s) return s;
        k_macro_scatter_x4<<<g3, 128, 0, st>>>(g.nx, cy, cz, (const float*)p->Hc, (float*)Hs_dev, accumulate);
    } else if (p->prec == DEMAG_FP32) {
        k_macro_avg<float><<<ga, 256, 0, st>>>(g.nx, g.ny, g.nz, cx, cy, cz, (const float*)S_dev, (float*)p->Mc, f);
        s = apply_outer<float>(p, (const float*)p->Mc, (float*)p->Hc, st);
        if (s) return s;
        k_macro_scatter<float><<<gs, 256, 0, st>>>(g.nx, g.ny, g.nz, cx, cy, cz, (const float*)p->Hc, (float*)Hs_dev, accumulate);
    } else {
        k_macro_avg<double><<<ga, 256, 0, st>>>(g.nx, g.ny, g.nz, cx, cy, cz, (const double*)S_dev, (double*)p->Mc, f);
        s = apply_outer<double>(p, (const double*)p->Mc, (double*)p->Hc, st);
        if (s) return s;
        k_macro_scatter<double><<<gs, 256, 0, st>>>(g.nx, g.ny, g.nz, cx, cy, cz, (const double*)p->Hc, (double*)Hs_dev, accumulate);
    }
    CUDA_TRY(cudaGetLastError());
    return DEMAG_OK;
}

// ================================================================================ no-allocation atomistic entry point
// For callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid it):
// demag_apply_atomistic with its two macrocell arrays (M and H on the plan's mesh, the scratch that
// demag_atomistic_reserve would allocate) taken from ONE file-scope device array of fixed size instead.
//   * Every GPU that loads this library holds the DEMAG_STATIC_SCRATCH_BYTES (16 MiB) of the array until the process exits.
//   * In host code `g_static_scratch` is only a stand-in for the symbol, NOT a device address: its device address is
//     resolved with cudaGetSymbolAddress once per device (with that device current) and cached; kernels get that pointer.
//   * All calls share the array and it keeps the last call's contents.  Nothing in it has to start at zero: the
//     average kernel writes every cell of M and the convolution writes every cell of H before the scatter reads it.
//   * Calls that overlap on the GPU (two streams, two plans, two threads) race on the array: serialise them.
namespace {
constexpr size_t kStaticScratchBytes = DEMAG_STATIC_SCRATCH_BYTES;
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];
constexpr int kMaxDevices = 64;
void* g_static_scratch_addr[kMaxDevices] = {};     // device address of g_static_scratch on each device (NULL: not resolved yet)

demag_status static_scratch_ptr(int device, void** out)
{
    if (device < 0 || device >= kMaxDevices) return fail(DEMAG_ERR_UNSUPPORTED, "device %d: the static scratch serves devices 0..%d", device, kMaxDevices - 1);
    void* q = __atomic_load_n(&g_static_scratch_addr[device], __ATOMIC_ACQUIRE);
    if (!q) {      // set-up, once per device, with that device current (the caller checked): no allocation involved
        cudaError_t e = cudaGetSymbolAddress(&q, g_static_scratch);
        if (e != cudaSuccess || !q) return fail(DEMAG_ERR_CUDA, "cudaGetSymbolAddress(static scratch): %s", cudaGetErrorString(e));
        __atomic_store_n(&g_static_scratch_addr[device], q, __ATOMIC_RELEASE);
    }
    *out = q;
    return DEMAG_OK;
}
}  // namespace

extern "C" size_t demag_static_scratch_bytes(void) { return kStaticScratchBytes; }

extern "C" demag_status demag_apply_atomistic_static(demag_plan_t p, const void* S_dev, void* Hs_dev, int cx, int cy, int cz,
                                                     double mu_s_in_muB, double a, int accumulate, void* cuda_stream)
{
    g_err[0] = 0;
    if (!p) return fail(DEMAG_ERR_INVALID_ARG, "plan is NULL");
    if (cx < 1 || cy < 1 || cz < 1 || !(a > 0) || !isfinite(mu_s_in_muB))
        return fail(DEMAG_ERR_INVALID_ARG, "bad macrocell / lattice arguments");
    struct { int nx, ny, nz; } g = {p->on[0], p->on[1], p->on[2]};     // the caller's macrocell mesh
    const double want[3] = {cx * a, cy * a, cz * a};
    for (int i = 0; i < 3; ++i)
        if (fabs(want[i] - p->h[i]) > 1e-9 * p->h[i])
            return fail(DEMAG_ERR_INVALID_ARG, "plan cell size must equal macrocell size c*a (axis %d)", i);
    const size_t nc = (size_t)g.nx * g.ny * g.nz;
    const size_t half = (3 * nc * p->esz + 255) / 256 * 256;          // M at offset 0, H at offset `half`
    if (2 * half > kStaticScratchBytes)
        return fail(DEMAG_ERR_UNSUPPORTED, "mesh %d x %d x %d needs %zu bytes of macrocell scratch, the static array holds %zu "
                    "(at most %zu cells in this precision): use demag_atomistic_reserve + demag_apply_atomistic",
                    g.nx, g.ny, g.nz, 2 * half, kStaticScratchBytes, kStaticScratchBytes / (6 * p->esz));
    const size_t nspin3 = (size_t)3 * g.nx * cx * g.ny * cy * g.nz * cz;
    demag_status s = check_apply_args(p, S_dev, Hs_dev, nspin3 * p->esz);      // incl. "the plan's device is the current device"
    if (s) return s;
    if (!p->has_kernel) return fail(DEMAG_ERR_NO_KERNEL, "demag_set_kernel has not been called");
    void* base = nullptr;
    if ((s = static_scratch_ptr(p->device, &base))) return s;
    void* Mc = base;
    void* Hc = (unsigned char*)base + half;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const double muB = 9.2740100783e-24;
    const double f = muB * mu_s_in_muB / ((double)cx * cy * cz * a * a * a);
    const unsigned ga = (unsigned)std::min<size_t>((3 * nc + 255) / 256, (size_t)1 << 22);
    const unsigned gs = (unsigned)std::min<size_t>((nspin3 / 4 + 255) / 256 + 1, (size_t)p->sm_count * 32);
    if (p->prec == DEMAG_FP32 && cx == 4 && g.ny <= 65535 && 3 * g.nz <= 65535) {
        const dim3 g3((unsigned)((g.nx + 127) / 128), (unsigned)g.ny, (unsigned)(3 * g.nz));
        k_macro_avg_x4<<<g3, 128, 0, st>>>(g.nx, cy, cz, (const float*)S_dev, (float*)Mc, f);
        s = apply_outer<float>(p, (const float*)Mc, (float*)Hc, st);
        if (s) return s;
        k_macro_scatter_x4<<<g3, 128, 0, st>>>(g.nx, cy, cz, (const float*)Hc, (float*)Hs_dev, accumulate);
    } else if (p->prec == DEMAG_FP32) {
        k_macro_avg<float><<<ga, 256, 0, st>>>(g.nx, g.ny, g.nz, cx, cy, cz, (const float*)S_dev, (float*)Mc, f);
        s = apply_outer<float>(p, (const float*)Mc, (float*)Hc, st);
        if (s) return s;
        k_macro_scatter<float><<<gs, 256, 0, st>>>(g.nx, g.ny, g.nz, cx, cy, cz, (const float*)Hc, (float*)Hs_dev, accumulate);
    } else {
        k_macro_avg<double><<<ga, 256, 0, st>>>(g.nx, g.ny, g.nz, cx, cy, cz, (const double*)S_dev, (double*)Mc, f);
        s = apply_outer<double>(p, (const double*)Mc, (double*)Hc, st);
        if (s) return s;
        k_macro_scatter<double><<<gs, 256, 0, st>>>(g.nx, g.ny, g.nz, cx, cy, cz, (const double*)Hc, (double*)Hs_dev, accumulate);
    }
    CUDA_TRY(cudaGetLastError());
    return DEMAG_OK;
}
