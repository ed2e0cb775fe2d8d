// llg.cu -- minimal consumer of the convolution: the LLG equation (Eq. (5)) integrated with RK4, the
// demagnetizing field of the sub-steps either convolved or extrapolated from previously computed fields.
// Everything goes through the public C ABI of include/demag.h (demag_apply, demag_extrapolate): this file knows nothing
// about the plan's internals.  SURVEY.md 8(f) row 4; readings R20-R22 of DESIGN.md.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <new>

#include "../../include/demag.h"

extern "C" void demag_set_last_error_(const char* msg);

namespace {

demag_status fail(demag_status st, const char* msg) { demag_set_last_error_(msg); return st; }

constexpr int kKeep = 5;          // quartic: five kept fields ("the RK4 method requires a quartic polynomial")

// One RK4 stage for every cell, fused: K = f(Min, Hd + Hzee);  acc (+)= wdt K;  Mout = M0 + cdt K  (stages 1-3) or
// M0 += acc + wdt K (stage 4).  Planar [3][n] arrays.  STAGE 1: Min == M0, acc is written; STAGE 4: M0 is updated.
template <typename T, int STAGE>
__global__ void __launch_bounds__(256) k_llg_stage(size_t n, T* __restrict__ M0, const T* __restrict__ Min, const T* __restrict__ Hd,
                                                   T* __restrict__ Mout, T* __restrict__ acc, T hx, T hy, T hz, T gp, T aoms, T cdt, T wdt)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const T mx = Min[i], my = Min[n + i], mz = Min[2 * n + i];
        const T ex = Hd[i] + hx, ey = Hd[n + i] + hy, ez = Hd[2 * n + i] + hz;
        const T tx = my * ez - mz * ey, ty = mz * ex - mx * ez, tz = mx * ey - my * ex;               // M x H
        const T ux = my * tz - mz * ty, uy = mz * tx - mx * tz, uz = mx * ty - my * tx;               // M x (M x H)
        const T kx = gp * (tx + aoms * ux), ky = gp * (ty + aoms * uy), kz = gp * (tz + aoms * uz);   // dM/dt
        if (STAGE == 4) {
            M0[i] += acc[i] + wdt * kx; M0[n + i] += acc[n + i] + wdt * ky; M0[2 * n + i] += acc[2 * n + i] + wdt * kz;
        } else {
            const T bx = STAGE == 1 ? mx : M0[i], by = STAGE == 1 ? my : M0[n + i], bz = STAGE == 1 ? mz : M0[2 * n + i];
            if (STAGE == 1) { acc[i] = wdt * kx; acc[n + i] = wdt * ky; acc[2 * n + i] = wdt * kz; }
            else { acc[i] += wdt * kx; acc[n + i] += wdt * ky; acc[2 * n + i] += wdt * kz; }
            Mout[i] = bx + cdt * kx; Mout[n + i] = by + cdt * ky; Mout[2 * n + i] = bz + cdt * kz;
        }
    }
}

template <typename T>
__global__ void __launch_bounds__(256) k_mean3(size_t n, const T* __restrict__ M, double inv_n, double* __restrict__ out)
{
    double s[3] = {0.0, 0.0, 0.0};
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        s[0] += (double)M[i]; s[1] += (double)M[n + i]; s[2] += (double)M[2 * n + i];
    }
    __shared__ double sh[3][8];
    for (int c = 0; c < 3; ++c) {
        double v = s[c];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0) sh[c][threadIdx.x >> 5] = v;
    }
    __syncthreads();
    if (threadIdx.x < 3) {
        double v = 0.0;
        for (int w = 0; w < 8; ++w) v += sh[threadIdx.x][w];
        atomicAdd(out + threadIdx.x, v * inv_n);
    }
}

}  // namespace

struct demag_llg_s {
    demag_plan_t plan = nullptr;
    int prec = 0, sm_count = 1;
    size_t n = 0, bytes = 0;            // cells, bytes of one [3][n] field
    double Ms = 0, alpha = 0, gamma = 0, Hz[3] = {0, 0, 0};
    void* Mst = nullptr; void* acc = nullptr; void* Hsub = nullptr;
    void* hist[kKeep] = {};             // ring of the fields convolved at the start of the last steps
    double thist[kKeep] = {};
    int nhist = 0, head = 0;
    double t = 0;
    long long nconv = 0, nextrap = 0;
};

namespace {

template <typename T>
demag_status step_impl(demag_llg_s* L, T* M, double dt, bool extrapolate, cudaStream_t st)
{
    const unsigned grid = (unsigned)((L->n + 255) / 256 < (size_t)L->sm_count * 16 ? (L->n + 255) / 256 : (size_t)L->sm_count * 16);
    const T hx = (T)L->Hz[0], hy = (T)L->Hz[1], hz = (T)L->Hz[2];
    const T gp = (T)(-L->gamma / (1.0 + L->alpha * L->alpha)), aoms = (T)(L->alpha / L->Ms);
    T* Mst = (T*)L->Mst; T* acc = (T*)L->acc; T* Hsub = (T*)L->Hsub;
    // stage 1: the field at the start of the step is always convolved, straight into the ring of kept fields
    const int slot = L->head;
    demag_status s = demag_apply(L->plan, M, L->hist[slot], st);
    if (s) return s;
    L->nconv++;
    L->thist[slot] = L->t;
    L->head = (L->head + 1) % kKeep;
    if (L->nhist < kKeep) L->nhist++;
    const bool use = extrapolate && L->nhist == kKeep;
    auto field = [&](const T* X, double ts, bool same_as_last) -> demag_status {
        if (use) {
            if (same_as_last) return DEMAG_OK;                      // stages 2 and 3 share the time t + dt/2
            L->nextrap++;
            return demag_extrapolate(L->plan, kKeep, (const void* const*)L->hist, L->thist, ts, Hsub, 0, st);
        }
        L->nconv++;
        return demag_apply(L->plan, X, Hsub, st);
    };
    k_llg_stage<T, 1><<<grid, 256, 0, st>>>(L->n, M, M, (const T*)L->hist[slot], Mst, acc, hx, hy, hz, gp, aoms, (T)(0.5 * dt), (T)(dt / 6.0));
    if ((s = field(Mst, L->t + 0.5 * dt, false))) return s;
    k_llg_stage<T, 2><<<grid, 256, 0, st>>>(L->n, M, Mst, Hsub, Mst, acc, hx, hy, hz, gp, aoms, (T)(0.5 * dt), (T)(dt / 3.0));
    if ((s = field(Mst, L->t + 0.5 * dt, true))) return s;
    k_llg_stage<T, 3><<<grid, 256, 0, st>>>(L->n, M, Mst, Hsub, Mst, acc, hx, hy, hz, gp, aoms, (T)dt, (T)(dt / 3.0));
    if ((s = field(Mst, L->t + dt, false))) return s;
    k_llg_stage<T, 4><<<grid, 256, 0, st>>>(L->n, M, Mst, Hsub, Mst, acc, hx, hy, hz, gp, aoms, (T)0, (T)(dt / 6.0));
    L->t += dt;
    if (cudaGetLastError() != cudaSuccess) return fail(DEMAG_ERR_CUDA, "demag_llg_step: kernel launch failed");
    return DEMAG_OK;
}

}  // namespace

extern "C" {

demag_status demag_llg_create(demag_llg_t* out, demag_plan_t plan, double Ms, double alpha, double gamma)
{
    if (!out) return fail(DEMAG_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!plan) return fail(DEMAG_ERR_INVALID_ARG, "plan is NULL");
    if (!(Ms > 0) || !(alpha >= 0) || !(gamma > 0) || !isfinite(Ms) || !isfinite(alpha) || !isfinite(gamma))
        return fail(DEMAG_ERR_INVALID_ARG, "Ms and gamma must be positive, alpha non-negative, all finite");
    int nx, ny, nz, prec;
    demag_status s = demag_plan_dims(plan, &nx, &ny, &nz, &prec);
    if (s) return s;
    demag_llg_s* L = new (std::nothrow) demag_llg_s();
    if (!L) return fail(DEMAG_ERR_ALLOC, "out of host memory");
    L->plan = plan; L->prec = prec; L->Ms = Ms; L->alpha = alpha; L->gamma = gamma;
    L->n = (size_t)nx * ny * nz;
    L->bytes = 3 * L->n * (prec == DEMAG_FP32 ? 4 : 8);
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&L->sm_count, cudaDevAttrMultiProcessorCount, dev);
    void** all[3 + kKeep] = {&L->Mst, &L->acc, &L->Hsub, &L->hist[0], &L->hist[1], &L->hist[2], &L->hist[3], &L->hist[4]};
    for (void** q : all)
        if (cudaMalloc(q, L->bytes) != cudaSuccess) { demag_llg_destroy(L); return fail(DEMAG_ERR_ALLOC, "demag_llg_create: out of device memory"); }
    *out = L;
    return DEMAG_OK;
}

demag_status demag_llg_set_field(demag_llg_t L, double Hx, double Hy, double Hz)
{
    if (!L) return fail(DEMAG_ERR_INVALID_ARG, "integrator is NULL");
    if (!isfinite(Hx) || !isfinite(Hy) || !isfinite(Hz)) return fail(DEMAG_ERR_INVALID_ARG, "field is not finite");
    L->Hz[0] = Hx; L->Hz[1] = Hy; L->Hz[2] = Hz;
    return DEMAG_OK;
}

demag_status demag_llg_step(demag_llg_t L, void* M_dev, double dt, int extrapolate, void* cuda_stream)
{
    if (!L || !M_dev) return fail(DEMAG_ERR_INVALID_ARG, "NULL argument");
    if (!(dt > 0) || !isfinite(dt)) return fail(DEMAG_ERR_INVALID_ARG, "dt must be positive and finite");
    if ((uintptr_t)M_dev & 15) return fail(DEMAG_ERR_INVALID_ARG, "device pointers must be 16-byte aligned");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    return L->prec == DEMAG_FP32 ? step_impl<float>(L, (float*)M_dev, dt, extrapolate != 0, st)
                                 : step_impl<double>(L, (double*)M_dev, dt, extrapolate != 0, st);
}

demag_status demag_llg_mean(demag_llg_t L, const void* M_dev, double* mean3_dev, void* cuda_stream)
{
    if (!L || !M_dev || !mean3_dev) return fail(DEMAG_ERR_INVALID_ARG, "NULL argument");
    if ((uintptr_t)mean3_dev & 7) return fail(DEMAG_ERR_INVALID_ARG, "mean3_dev must be 8-byte aligned");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (cudaMemsetAsync(mean3_dev, 0, 3 * sizeof(double), st) != cudaSuccess) return fail(DEMAG_ERR_CUDA, "demag_llg_mean: memset failed");
    const unsigned grid = (unsigned)((L->n + 255) / 256 < (size_t)L->sm_count * 8 ? (L->n + 255) / 256 : (size_t)L->sm_count * 8);
    if (L->prec == DEMAG_FP32) k_mean3<float><<<grid, 256, 0, st>>>(L->n, (const float*)M_dev, 1.0 / (double)L->n, mean3_dev);
    else k_mean3<double><<<grid, 256, 0, st>>>(L->n, (const double*)M_dev, 1.0 / (double)L->n, mean3_dev);
    if (cudaGetLastError() != cudaSuccess) return fail(DEMAG_ERR_CUDA, "demag_llg_mean: kernel launch failed");
    return DEMAG_OK;
}

demag_status demag_llg_counts(demag_llg_t L, long long* n_convolutions, long long* n_extrapolations, double* time)
{
    if (!L) return fail(DEMAG_ERR_INVALID_ARG, "integrator is NULL");
    if (n_convolutions) *n_convolutions = L->nconv;
    if (n_extrapolations) *n_extrapolations = L->nextrap;
    if (time) *time = L->t;
    return DEMAG_OK;
}

demag_status demag_llg_reset(demag_llg_t L)
{
    if (!L) return fail(DEMAG_ERR_INVALID_ARG, "integrator is NULL");
    L->nhist = 0; L->head = 0; L->t = 0; L->nconv = 0; L->nextrap = 0;
    return DEMAG_OK;
}

demag_status demag_llg_destroy(demag_llg_t L)
{
    if (!L) return DEMAG_OK;
    cudaFree(L->Mst); cudaFree(L->acc); cudaFree(L->Hsub);
    for (void* q : L->hist) cudaFree(q);
    delete L;
    return DEMAG_OK;
}

}  // extern "C"
