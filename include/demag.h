/*
 * demag.h -- C ABI of the B200-native demagnetizing-field convolution.
 *
 * Computes, on ONE GPU, the long-range demagnetizing field of arXiv 2308.08447, Eq. (1)
 * (Section II):
 *
 *        H_d,i = - sum_j N(i-j) M_j        (sum over all cells j of the mesh, j = i included)
 *
 * evaluated as a zero-padded 3D FFT convolution (Appendix A :228-343):
 * x R2C FFT -> y FFT -> z FFT -> multiply with the transformed tensor -> inverse z, y -> x C2R.
 *
 * Conventions (readings R3, R6, R8):
 *   - mesh of nx*ny*nz cuboid cells of size hx*hy*hz metres, 1 <= nx <= 8192, 1 <= ny, nz <= 4096;
 *   - an axis is zero-padded to N_a = 2 m_a, m_a = the next power of two >= n_a (an exact linear convolution needs
 *     N_a >= 2 n_a - 1), unless n_a == 1 or its PBC flag is set (then N_a = n_a, and a periodic
 *     n_a must itself be a power of two).  A mesh whose sizes are not all powers of two is embedded, with zeros,
 *     in the m_x*m_y*m_z mesh inside the plan (two extra copies per apply, same result);
 *   - M, H: planar device arrays [3][nz][ny][nx], x fastest, components x,y,z, in A/m,
 *     float (DEMAG_FP32) or double (DEMAG_FP64), 16-byte aligned, not aliased;
 *   - tensor component order: xx, yy, zz, xy, xz, yz; N is dimensionless;
 *   - pointers named *_dev are device pointers, *_host are host pointers;
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = default stream);
 *   - every function returns a demag_status; no exceptions, no abort, no printing.
 *
 * Ownership: the plan owns its workspace, twiddle tables and kernel spectrum (allocated in
 * demag_plan_create / demag_set_kernel).  The caller owns M, H, S, Hs, E.
 * demag_apply / demag_energy / demag_apply_atomistic never allocate, never synchronise, never touch
 * the host: they only enqueue kernels on `cuda_stream`.  A plan is not re-entrant (one apply in
 * flight per plan).
 */
#ifndef DEMAG_H_
#define DEMAG_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct demag_plan_s* demag_plan_t;            /* opaque; owned by the library */

typedef enum {
    DEMAG_OK = 0,
    DEMAG_ERR_INVALID_ARG = 1,   /* NULL / misaligned / aliased pointer, non-positive size          */
    DEMAG_ERR_UNSUPPORTED = 2,   /* size above the limits, periodic size not a power of two, built-in tensor + PBC,
                                    fp64 with nz > 2048 (an 8192-point fp64 z line exceeds shared memory)   */
    DEMAG_ERR_ALLOC = 3,         /* cudaMalloc / malloc failed                                       */
    DEMAG_ERR_CUDA = 4,          /* a CUDA runtime call or launch failed (see demag_last_error)      */
    DEMAG_ERR_NO_KERNEL = 5      /* demag_apply before demag_set_kernel                              */
} demag_status;

enum { DEMAG_FP32 = 0, DEMAG_FP64 = 1 };                 /* precision of M, H, workspace, spectrum */
enum { DEMAG_PBC_X = 1, DEMAG_PBC_Y = 2, DEMAG_PBC_Z = 4 };  /* pbc_flags bitmask     */

/* Create a plan for an nx*ny*nz mesh of hx*hy*hz [m] cells (the statement of the
 * problem; :31-35 padding; :47 PBC axes are not padded).  Allocates workspace and FFT tables on the
 * current CUDA device.  *out is set to NULL on failure. */
demag_status demag_plan_create(demag_plan_t* out, int nx, int ny, int nz,
                               double hx, double hy, double hz,
                               unsigned pbc_flags, int precision);

/* Compute and store the transformed tensor ("convolution kernel ... computed in the initialization
 * stage"; stored packed by its y/z symmetries as real arrays).
 *   N6_host == NULL: built-in fp64 Newell builder on the GPU ("formulas in Ref. [23]";
 *                    DESIGN.md R1, R4).  With PBC flags: the periodic tensor of demag_set_pbc_images.
 *   N6_host != NULL: host array double[6][nz][ny][nx]: N_c at the non-negative cell offsets
 *                    (dx,dy,dz); negative offsets follow by parity (diagonal even; xy odd in x,y;
 *                    xz odd in x,z; yz odd in y,z).  On a PBC axis the n_a entries are the periodic
 *                    kernel at offsets 0..n_a-1 (no parity folding on that axis); a periodic kernel obeys
 *                    K(n_a - d) = parity * K(d) there, and only that symmetric part of the table is used
 *                    (the stored spectrum is real).
 * The spectrum is computed in fp64, the factor -1/(Nx Ny Nz) is folded in (R3), and it is
 * rounded once to fp32 (kept fp64 for a DEMAG_FP64 plan).  Synchronous (plan-time call). */
demag_status demag_set_kernel(demag_plan_t plan, const double* N6_host);

/* Built-in periodic tensor ("modified convolution kernel"; the paper's reference [25] is not available,
 * DESIGN.md R11 states the reading): on every periodic axis a the open-boundary tensor is summed over `images` periodic
 * images on each side, T(d) = sum_{|m_a| <= images} N((d_a + m_a n_a) h_a), and symmetrised under d_a -> n_a - d_a
 * (indices mod n_a; a periodic kernel is symmetric up to the component's parity, the truncated sum only up to its
 * last images), which for d_a > 0 amounts to weight 1/2 on the images m_a = -images-1 and m_a = images.  Default 10; 0..1000.  Takes effect at the
 * next demag_set_kernel(plan, NULL) / demag_get_kernel_real.  Cost grows with (2 images + 2)^(periodic axes). */
demag_status demag_set_pbc_images(demag_plan_t plan, int images);

/* H = -N * M  (Eq. (1); execution order of Appendix A).
 * M_dev, H_dev: device arrays [3][nz][ny][nx] of the plan's precision.  Asynchronous on the stream.
 * M is not modified; H is overwritten.  DEMAG_ERR_NO_KERNEL before demag_set_kernel. */
demag_status demag_apply(demag_plan_t plan, const void* M_dev, void* H_dev, void* cuda_stream);

/* H_eff += -N * M: the same convolution, ADDED into an existing effective-field array (the demagnetizing
 * field is one contribution to H_eff) inside the last kernel, so the integrator needs no extra pass over H.
 * Same arguments, layout and errors as demag_apply; Heff_dev is read and written. */
demag_status demag_apply_add(demag_plan_t plan, const void* M_dev, void* Heff_dev, void* cuda_stream);

/* Polynomial extrapolation of the demagnetizing field at sub-steps of the time integrator ("polynomial
 * extrapolation of the demagnetizing field at sub-steps of the higher order evaluation method, using previously computed
 * values ... the RK4 method requires a quartic polynomial, whilst the RKF56 method requires a quintic polynomial";
 * DESIGN.md R19): the polynomial of degree npts-1 through the npts previously computed fields, evaluated at time t,
 *     H(t) = sum_k L_k(t) H_k,   L_k(t) = prod_{j != k} (t - t_j) / (t_k - t_j)        (every array entry on its own),
 * written to H_out_dev (accumulate == 0) or added to it (accumulate != 0: H_out is then H_eff), in ONE streaming pass
 * that replaces a whole convolution at that sub-step.
 *   H_hist_dev:  host array of npts device pointers, each [3][nz][ny][nx] of the plan's precision (this rank's rows for a
 *                sharded plan), 16-byte aligned, none overlapping H_out_dev;   1 <= npts <= 8 (quartic: 5, quintic: 6).
 *   t_hist_host: host array of the npts distinct sample times; t: the time wanted (any unit, only ratios enter).
 * The weights are evaluated on the host in extended precision; the device sums in the plan's precision with FMAs.
 * Asynchronous on the stream; the host arrays are read before the call returns. */
demag_status demag_extrapolate(demag_plan_t plan, int npts, const void* const* H_hist_dev, const double* t_hist_host,
                               double t, void* H_out_dev, int accumulate, void* cuda_stream);

/* Demagnetizing energy  E = -(mu0/2) hx hy hz sum_i M_i . H_i  [J] (R12), accumulated in
 * fp64 and written to the device scalar *E_dev (double).  Asynchronous on the stream. */
demag_status demag_energy(demag_plan_t plan, const void* M_dev, const void* H_dev,
                          double* E_dev, void* cuda_stream);

/* Atomistic front end (Eq. (9)): unit spins S_dev [3][Lz][Ly][Lx] on a simple cubic
 * lattice (constant a [m], moment mu_s_in_muB Bohr magnetons) are averaged into macrocells of
 * cx*cy*cz spins, M = mu_B mu_s sum(S^) / (cx cy cz a^3); the plan's convolution is applied; the
 * cell field is written to every spin of the cell, Hs_dev [3][Lz][Ly][Lx] (overwritten if
 * accumulate == 0, added to if accumulate != 0).  The spin lattice is (nx*cx, ny*cy, nz*cz); the plan
 * must have been created with h_a = c_a * a (checked to 1e-9 relative).
 * The two macrocell arrays (M and H on the plan's mesh) live in the plan and are allocated by
 * demag_atomistic_reserve, NOT by this call: without them it returns DEMAG_ERR_INVALID_ARG.  Like demag_apply it never
 * allocates or synchronises, so its first call can already be captured in a CUDA graph. */
demag_status demag_apply_atomistic(demag_plan_t plan, const void* S_dev, void* Hs_dev,
                                   int cx, int cy, int cz, double mu_s_in_muB, double a,
                                   int accumulate, void* cuda_stream);

/* Allocate the macrocell arrays demag_apply_atomistic works on (2 * 3 * nx*ny*nz reals; counted by
 * demag_workspace_bytes from then on).  Idempotent; synchronous (cudaMalloc); DEMAG_ERR_ALLOC if out of memory. */
demag_status demag_atomistic_reserve(demag_plan_t plan);

/* demag_apply_atomistic for callers that cannot call cudaMalloc at all (code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid it): the same three steps (Eq. (9) average, the plan's convolution, scatter), with
 * the two macrocell arrays taken from one file-scope device array of DEMAG_STATIC_SCRATCH_BYTES inside the library instead of
 * from demag_atomistic_reserve.  Same arguments, same result bit for bit.  It calls no cudaMalloc / cudaFree / allocating
 * routine; its first call on a device resolves the array's device address (cudaGetSymbolAddress, no allocation).
 *   - Limit: 2 * 3 * nx*ny*nz reals (each half rounded up to 256 bytes) must fit: at most 699,050 cells in fp32, 349,525 in
 *     fp64; larger meshes return DEMAG_ERR_UNSUPPORTED (use demag_atomistic_reserve + demag_apply_atomistic).
 *   - Every GPU that loads the library holds the array until the process exits.
 *   - All calls of all plans share the array, which keeps the last call's contents (nothing in it needs clearing: both halves
 *     are fully overwritten before they are read).  Calls that OVERLAP on the GPU (different streams or threads) race on it:
 *     serialise them on one stream. */
#define DEMAG_STATIC_SCRATCH_BYTES (16u << 20)
demag_status demag_apply_atomistic_static(demag_plan_t plan, const void* S_dev, void* Hs_dev,
                                          int cx, int cy, int cz, double mu_s_in_muB, double a,
                                          int accumulate, void* cuda_stream);
size_t demag_static_scratch_bytes(void);      /* = DEMAG_STATIC_SCRATCH_BYTES of the loaded library */

/* Copy back the REAL-SPACE tensor the plan was given or built: double[6][nz][ny][nx] (host).
 * For builder-vs-oracle parity tests.  Synchronous. */
demag_status demag_get_kernel_real(demag_plan_t plan, double* N6_host);

/* Bytes of device memory the plan holds (workspace + tables + kernel spectrum). */
size_t demag_workspace_bytes(demag_plan_t plan);

/* Tuning knob: how many kx planes one L2-resident slab of the y/z stages covers (0 = automatic).
 * Does not change results. */
demag_status demag_set_slab(demag_plan_t plan, int kx_per_slab);

/* Instrumentation (not the hot path): runs one demag_apply on the stream with a CUDA event pair around
 * every kernel launch, synchronises, and writes the summed device time in milliseconds of each stage to
 * stage_ms_host[5] = { x R2C, y forward, z forward*multiply*z inverse, y inverse, x C2R }
 * (Appendix A execution order) and the launch count of each stage to
 * stage_launches_host[5] (either pointer may be NULL).  Same arguments and result as demag_apply. */
demag_status demag_apply_profiled(demag_plan_t plan, const void* M_dev, void* H_dev, void* cuda_stream,
                                  float* stage_ms_host, int* stage_launches_host);

/* Number of kernel launches one demag_apply enqueues with the current settings. */
int demag_launches_per_apply(demag_plan_t plan);

/* Which kernel family demag_apply uses for this plan: 1 = the compile-time specialised two-lines-per-thread
 * kernels (DEMAG_FP32 plans with all axes zero padded and sizes in their instantiated range), 0 = the size-generic
 * kernels.  Both compute the same convolution (Appendix A).  The environment variable DEMAG_PATH,
 * read by demag_plan_create, overrides the choice: "generic" forces 0, "fast" also admits DEMAG_FP64 plans to 1
 * (used by the tests to cover both families in both precisions). */
int demag_path(demag_plan_t plan);

/* ---------------------------------------------------------------------------------------------------------------
 * Several GPUs, one process (rank) per GPU: the paper's multi-GPU convolution (Fig. 1; Appendix A,
 * PAPER.md:261-341), DESIGN.md 8.
 *
 * Partitioning.  The paper splits M / H along x and needs four transfers per convolution (M->In, S1->S2, S2->S1,
 * Out->H).  Here M and H are split along Y -- rank r owns the rows [y0_r, y0_r + ny_r) of every
 * (component, z) plane, arrays [3][nz][ny_r][nx] -- so the x transforms are local and only the two spectrum
 * transfers remain (12 n_c (G-1)/G^2 reals per rank instead of the paper's 18).  The y and z stages and
 * the stored kernel use the paper's x partitioning of the half spectrum ("for the y and z FFT steps the
 * x dimension partitioning is used"; K^(g)): rank s owns the frequency pairs (k, nx-k),
 * k in [q0_s, q0_s + nq_s), of 0 <= k <= nx/2.  Both splits give every rank `per` units and the last rank the
 * remainder, see demag_shard_range.
 * The transfers are not copies: the x R2C kernel stores every spectrum element directly into the workspace of the
 * rank that owns its pair, and the y inverse kernel stores every cropped element into the workspace of the rank
 * that owns its row (peer device pointers, NVLink), so the exchange overlaps the transforms tile by tile.
 *
 * Protocol per convolution, on every rank, all on one stream:
 *     demag_apply_sharded(plan, 0, M_loc, NULL, stream);     x R2C            (writes peers' W1in)
 *     <barrier over all ranks, ordered on the stream>
 *     demag_apply_sharded(plan, 1, NULL, NULL, stream);      y FFT, z FFT . multiply . z IFFT, y IFFT (writes peers' W1out)
 *     <barrier over all ranks, ordered on the stream>
 *     demag_apply_sharded(plan, 2, NULL, H_loc, stream);     x C2R
 * The barrier is the caller's (the Python binding enqueues an NCCL all-reduce of one element on the same stream).  No
 * barrier is needed between two convolutions.
 *
 * Restrictions (DEMAG_ERR_UNSUPPORTED otherwise): the fast kernel family only -- power-of-two mesh sizes, nz >= 2,
 * no periodic axis, sizes in the instantiated range (demag_path() == 1) -- world <= 16, and at least 16 rows
 * (8 for nx >= 1024 ... see demag_shard_range's align) and one frequency pair per rank. */

/* Host-only arithmetic of the partition: units [begin, begin + count) of n belong to `rank` of `world`; every rank
 * gets per = floor(n / world / align) * align units and the last one the remainder.  DEMAG_ERR_UNSUPPORTED if
 * per == 0, DEMAG_ERR_INVALID_ARG for bad arguments.  Needs no GPU. */
demag_status demag_shard_range(int n, int world, int rank, int align, int* begin, int* count);

/* As demag_plan_create, for rank `rank` of `world`; (nx, ny, nz) is the WHOLE mesh.  Allocates this rank's W1in,
 * W1out, its slab of the y/z workspace and, at demag_set_kernel (which takes the whole real-space table or NULL, as on
 * one GPU), only its part K^(rank) of the spectrum.  world == 1 is allowed (and equals demag_plan_create's result). */
demag_status demag_plan_create_sharded(demag_plan_t* out, int nx, int ny, int nz, double hx, double hy, double hz,
                                       unsigned pbc_flags, int precision, int rank, int world);

/* This rank's ranges (any pointer may be NULL): rows [y0, y0 + ny_loc), frequency pairs [q0, q0 + nq_loc). */
demag_status demag_shard_info(demag_plan_t plan, int* rank, int* world, int* y0, int* ny_loc, int* q0, int* nq_loc);

/* This rank's two exchange buffers (device pointers owned by the plan) and their sizes in bytes. */
demag_status demag_shard_buffers(demag_plan_t plan, void** w1in_dev, size_t* w1in_bytes, void** w1out_dev, size_t* w1out_bytes);

/* Wiring the ranks together.  Either exchange CUDA IPC handles between the processes:
 *   demag_shard_ipc_export writes 128 bytes (two cudaIpcMemHandle_t: W1in, W1out) to handles_host;
 *   demag_shard_ipc_connect takes world * 128 bytes, rank-major (an all-gather of the exports), opens every other
 *   rank's buffers (peer access over NVLink) and installs them;
 * or, when the buffers of all ranks are already addressable from this device (one process driving several plans),
 *   demag_shard_set_peers installs world pointers to the W1in and world pointers to the W1out buffers (host arrays
 *   of device pointers, entry `rank` must be the plan's own buffer).
 * DEMAG_ERR_INVALID_ARG for a plan that is not sharded; DEMAG_ERR_CUDA if a handle cannot be opened. */
demag_status demag_shard_ipc_export(demag_plan_t plan, void* handles_host);
demag_status demag_shard_ipc_connect(demag_plan_t plan, const void* all_handles_host);
demag_status demag_shard_set_peers(demag_plan_t plan, void* const* w1in_of_rank, void* const* w1out_of_rank);

/* One phase (0, 1, 2: see the protocol above) of the partitioned convolution.  M_loc_dev (phase 0) and H_loc_dev
 * (phase 2) are this rank's rows, [3][nz][ny_loc][nx] in the plan's precision, 16-byte aligned; the other pointer
 * arguments are ignored.  Asynchronous on the stream, never allocates or synchronises.
 * DEMAG_ERR_NO_KERNEL before demag_set_kernel, DEMAG_ERR_INVALID_ARG before the peers are installed, for a bad phase
 * or a plan that is not sharded.  demag_apply / demag_apply_add / demag_apply_atomistic on a sharded plan with
 * world > 1 return DEMAG_ERR_INVALID_ARG; demag_energy returns this rank's partial sum over its rows. */
demag_status demag_apply_sharded(demag_plan_t plan, int phase, const void* M_loc_dev, void* H_loc_dev, void* cuda_stream);

/* ---- Minimal time integrator that consumes the convolution: LLG equation, RK4, sub-step extrapolation ------------------
 * (only as far as needed to reproduce the error metric of PAPER.md:47.)
 *
 * Eq. (5):  dm/dt = -gamma m x H_eff + alpha m x dm/dt,  m = M / Ms,  H_eff = H_d + H_Zee  (the other
 * interaction fields of PAPER.md:94 are out of scope), solved for the derivative (R20):
 *     dM/dt = -gamma / (1 + alpha^2) [ M x H_eff + (alpha / Ms) M x (M x H_eff) ],
 * integrated with the classical 4th-order Runge-Kutta method, no renormalisation of |M| (R21).
 * H_d = -N * M is demag_apply of the plan.  With extrapolate != 0 (R22) it is convolved only at the START of
 * a step; the five most recent such fields are kept, and once five exist the fields of the three later stages (times
 * t + dt/2, t + dt/2, t + dt) are the quartic through them (demag_extrapolate): one convolution per step instead of four.
 *
 * The integrator owns eight field-sized work arrays (stage magnetisation, RK sum, sub-step field, five kept fields),
 * allocated in demag_llg_create; demag_llg_step only enqueues kernels on the stream (four fused stage kernels, one or
 * four convolutions, up to two extrapolation passes), never allocates, never synchronises.  gamma in m/(A s)
 * (mu0 |gamma_e| = 2.212761569e5), Ms and the fields in A/m, dt in seconds.  One-GPU plans only. */
typedef struct demag_llg_s* demag_llg_t;
demag_status demag_llg_create(demag_llg_t* out, demag_plan_t plan, double Ms, double alpha, double gamma);
/* Uniform applied field H_Zee (A/m); (0, 0, 0) after create. */
demag_status demag_llg_set_field(demag_llg_t llg, double Hx, double Hy, double Hz);
/* One RK4 step of size dt, in place on M_dev ([3][nz][ny][nx], plan precision, 16-byte aligned). */
demag_status demag_llg_step(demag_llg_t llg, void* M_dev, double dt, int extrapolate, void* cuda_stream);
/* Mesh average of M ("the average magnetization is recorded every time step"): mean3_dev[0..2] (double,
 * device), fp64 accumulation.  Asynchronous on the stream. */
demag_status demag_llg_mean(demag_llg_t llg, const void* M_dev, double* mean3_dev, void* cuda_stream);
/* Convolutions and extrapolation passes enqueued so far, and the integrator's time (any of the pointers may be NULL). */
demag_status demag_llg_counts(demag_llg_t llg, long long* n_convolutions, long long* n_extrapolations, double* time);
/* Forget the kept fields and set the time to zero (a new trajectory). */
demag_status demag_llg_reset(demag_llg_t llg);
demag_status demag_llg_destroy(demag_llg_t llg);

/* Mesh sizes (the caller's nx, ny, nz) and precision of a plan (any of the pointers may be NULL). */
demag_status demag_plan_dims(demag_plan_t plan, int* nx, int* ny, int* nz, int* precision);

/* Last error message of the calling thread ("" if none). */
const char* demag_last_error(void);

demag_status demag_plan_destroy(demag_plan_t plan);

#ifdef __cplusplus
}
#endif
#endif /* DEMAG_H_ */
