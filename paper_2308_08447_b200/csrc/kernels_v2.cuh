// kernels_v2.cuh -- the fast hot path of demag_apply: compile-time specialised kernels that process TWO lines
// per thread in packed fp32 (soa_core.cuh).  Same mathematics and execution order as kernels.cuh
// (x R2C -> y FFT -> z FFT . kernel multiplication . z IFFT -> y IFFT -> x C2R), different
// data layout of the private workspaces:
//
//   W1v [3][hq][nz][ny] quads   one quad = x-frequencies (k, Lc-k) of one (y,z): the pair the Hermitian split of
//                               the real transform produces / consumes together (hq = Lc/2 + 1, Lc = Nx/2 = nx)
//   W2v [3][nq][nz][Ny] quads   slab of nq pairs; y in the digit-reversed "position order" the forward passes
//                               leave behind (the stored kernel spectrum uses the same order: nothing is permuted)
//   Kv  [hq][kst][Nz/2+1][chunk][KT]    the six real components for the two frequencies of the pair, packed by
//                               symmetry in z AND y ((ny+1) x (nz+1) rows), -1/(Nx Ny Nz) and the
//                               1/2 of the real split folded in at plan time; split into 16-byte chunks and tiled by
//                               KT consecutive SLOTS (KT = the z kernel's tile width: a tile's rows are contiguous).
//                               Slots: W2v position py holds y frequency ky; the positions with
//                               ky <= Ny/2 are numbered in position order, a position with ky > Ny/2 uses the slot
//                               of Ny - ky with the sign of the y-odd components (xy, yz) flipped.  yslot[py] =
//                               slot | (mirrored << 31) is built at plan time for the y schedule in use, so that the
//                               columns of a tile (consecutive py) read consecutive slots (ascending or descending)
//
// Every kernel is templated on log2 of its transform length, its tile and its block size, so that every
// shared-memory offset is an immediate; twiddles come from per-pass tables (dup format, [m-1][lo]).
#pragma once
#include <cuda.h>          // CUtensorMap (type only: the encoder is fetched through the runtime, v2_host.cuh)
#include "soa_core.cuh"


namespace demag {
namespace v2 {

extern __shared__ __align__(32) unsigned char smem_v2[];

struct GeoV {
    int nx, ny, nz;      // mesh
    int Ny, Nz;          // padded (2 ny, 2 nz)
    int Lc;              // complex length of the packed real x transform = nx (Nx = 2 nx)
    int hq;              // number of (k, Lc-k) pairs = Lc/2 + 1
    int kpz;             // Nz/2 + 1
    int acc;             // x C2R: 0 = overwrite H, 1 = add into H (demag_apply_add)
    int trig;            // programmatic dependent launch: 0 = let the next grid in at block start, 1 = at block end
    int pf;              // L2 prefetch distance in blocks (0 = off): block b requests the input of tile b + pf
    int onx, ony, onz;   // the caller's mesh when it is embedded in the power-of-two mesh nx, ny, nz (R10): the x
                         // kernels read M / write H straight from / to the caller's arrays and supply the zeros themselves
    int pft;             // 1: the kernel's tensor map is valid -> the prefetch of a tile is ONE TMA request (pf_l2_tensor)
    int kst;             // slot tiles per pair plane of the stored kernel spectrum, ceil((Ny/2 + 1) / KT) (1 for one-cell-thick meshes)
};

template <typename T> struct TwSet { const CQ<T>* p[6]; };   // per-pass twiddle tables (NULL for stride-1 passes)

template <typename T> struct alignas(4 * sizeof(T)) KQ {     // kernel spectrum at one (q, kz', py): pairs over the two kx
    typename vec2<T>::type xx, yy, zz, xy, xz, yz;
};

// ---- partitioned workspaces (several GPUs; PAPER.md:31-35 and Fig. 1, :261-341) -------------------
// With G ranks the spectrum W1v exists twice, each copy split a different way (the paper's S1 and S2 partitionings):
//   W1in  on rank s: [3][nq_s][nz][ny]     all y of the pairs q this rank owns   (input of its y/z stage)
//   W1out on rank r: [3][hq][nz][ny_r]     all pairs of the rows y this rank owns (input of its x C2R stage)
// The kernel that PRODUCES a spectrum stores every element straight into the buffer of the rank that consumes it
// (peer-mapped device pointers over NVLink), so the paper's Transfer_S1_to_S2 / Transfer_S2_to_S1 (:272-289) happen
// inside the x R2C and y inverse kernels, tile by tile, and no pack / unpack copy exists.  Ranges are `per` units
// per rank, the last rank takes the remainder (:33 "approximately, since ... may not integer-divide").
constexpr int kMaxRanks = 16;
template <typename T> struct ShardMap {
    int G;                    // number of ranks
    int per;                  // units per rank: pairs q (x R2C -> W1in), rows y (y inverse -> W1out)
    int total;                // hq (x R2C), ny (y inverse)
    int off;                  // this rank's first global row y (x R2C), first global pair q (y inverse)
    int pitch;                // global ny (x R2C: row length of W1in), global hq (y inverse: pairs of W1out)
    CQ<T>* base[kMaxRanks];   // W1in / W1out of every rank, as seen from this device
};

// ---- 128-bit quad access ----------------------------------------------------------------------------
__device__ __forceinline__ CQ<float> ldq(const CQ<float>* p)
{
    const float4 v = *reinterpret_cast<const float4*>(p);
    CQ<float> r; r.re = make_float2(v.x, v.y); r.im = make_float2(v.z, v.w); return r;
}
__device__ __forceinline__ void stq(CQ<float>* p, CQ<float> a)
{
    *reinterpret_cast<float4*>(p) = make_float4(a.re.x, a.re.y, a.im.x, a.im.y);
}
__device__ __forceinline__ CQ<float> ldgq(const CQ<float>* p)
{
    const float4 v = __ldg(reinterpret_cast<const float4*>(p));
    CQ<float> r; r.re = make_float2(v.x, v.y); r.im = make_float2(v.z, v.w); return r;
}
__device__ __forceinline__ CQ<double> ldq(const CQ<double>* p)
{
    const double2* q = reinterpret_cast<const double2*>(p);
    CQ<double> r; r.re = q[0]; r.im = q[1]; return r;
}
__device__ __forceinline__ void stq(CQ<double>* p, CQ<double> a)
{
    double2* q = reinterpret_cast<double2*>(p);
    q[0] = a.re; q[1] = a.im;
}
__device__ __forceinline__ CQ<double> ldgq(const CQ<double>* p)
{
    const double2* q = reinterpret_cast<const double2*>(p);
    CQ<double> r; r.re = __ldg(q); r.im = __ldg(q + 1); return r;
}

// streaming global access of the field / workspace data (read once, written once per kernel): do not allocate in L1,
// which is left to the twiddle tables and the kernel spectrum
__device__ __forceinline__ CQ<float> ldsq(const CQ<float>* p)
{
    float4 v;
    asm volatile("ld.global.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    CQ<float> r; r.re = make_float2(v.x, v.y); r.im = make_float2(v.z, v.w); return r;
}
__device__ __forceinline__ CQ<double> ldsq(const CQ<double>* p)
{
    CQ<double> r;
    asm volatile("ld.global.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(r.re.x), "=d"(r.re.y) : "l"(p));
    asm volatile("ld.global.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(r.im.x), "=d"(r.im.y) : "l"(reinterpret_cast<const double2*>(p) + 1));
    return r;
}

// two adjacent quads (32 bytes, 32-byte aligned) in one 256-bit access (sm_100: LDG.256 / STG.256).  The x kernels move
// the two rows of a row pair this way: a warp's access then touches each 32-byte piece once instead of twice (half as
// many L1 wavefronts where the pieces of different threads lie in different lines: long rows, RP < 4).
template <bool NA> __device__ __forceinline__ void ldq2(const CQ<float>* p, CQ<float>& a, CQ<float>& b)
{
    float v[8];
    if (NA) asm volatile("ld.global.L1::no_allocate.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                         : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]) : "l"(p));
    else asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                      : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]) : "l"(p));
    a.re = make_float2(v[0], v[1]); a.im = make_float2(v[2], v[3]); b.re = make_float2(v[4], v[5]); b.im = make_float2(v[6], v[7]);
}
template <bool NA> __device__ __forceinline__ void ldq2(const CQ<double>* p, CQ<double>& a, CQ<double>& b)
{
    a = NA ? ldsq(p) : ldgq(p); b = NA ? ldsq(p + 1) : ldgq(p + 1);
}
__device__ __forceinline__ void stq2(CQ<float>* p, CQ<float> a, CQ<float> b)
{
    asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "f"(a.re.x), "f"(a.re.y), "f"(a.im.x), "f"(a.im.y),
                 "f"(b.re.x), "f"(b.re.y), "f"(b.im.x), "f"(b.im.y) : "memory");
}
__device__ __forceinline__ void stq2(CQ<double>* p, CQ<double> a, CQ<double> b) { stq(p, a); stq(p + 1, b); }

// ---- asynchronous bulk copy (TMA, 1D) signalled through an mbarrier -------------------------------------------
// Used by the long-line y kernel (one line pair per block, one block per SM): the next line lands in a staging
// buffer while the block transforms the current one.
// Programmatic dependent launch: the five kernels of one demag_apply are launched with
// cudaLaunchAttributeProgrammaticStreamSerialization (v2_host.cuh launch_pdl), so the blocks of kernel k+1 become resident
// while the last wave of kernel k drains.  Every kernel calls this before its first global access: it waits until the
// grid before it has completed and its stores are visible, then lets the grid after it be scheduled.  Without the
// launch attribute both instructions are no-ops.
__device__ __forceinline__ void pdl_enter(const GeoV& g)
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (!g.trig) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
// after the block's last global store (g.trig = 1: only the launch gap is hidden, no block of the next grid is
// resident while this one still works)
__device__ __forceinline__ void pdl_leave(const GeoV& g)
{
    if (g.trig) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// ---- L2 prefetch of a FUTURE tile's input --------------------------------------------------------------------
// The kernels hold 2-5 blocks of 2-8 warps per SM, each alternating between a load phase, shared-memory passes and a
// store phase: too few loads are in flight to cover the DRAM latency (ncu: "long scoreboard" is the top stall of all
// five kernels).  Blocks are dispatched in index order, so block b asks the memory system to bring the input of
// tile b + pf (pf ~ the number of co-resident blocks: the tile that starts when this one ends) into L2 while it
// works; that tile's loads then see the L2 latency instead of the DRAM latency.  Pure hint: no effect on results.
__device__ __forceinline__ void pf_l2_bulk(const void* p, uint32_t bytes)      // 16-byte aligned, bytes % 16 == 0
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}
__device__ __forceinline__ void pf_l2_line(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
// a whole strided tile (box of the kernel's tensor map) in one request: the TMA unit walks the rows, no LSU instruction
// per row (the per-row form costs the z kernel more than the prefetch gains when rows are 64-128 bytes)
__device__ __forceinline__ void pf_l2_tensor(const CUtensorMap* tm, int c0, int c1, int c2, int c3)
{
    asm volatile("cp.async.bulk.prefetch.tensor.4d.L2.global.tile [%0, {%1, %2, %3, %4}];"
                 ::"l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
// a span of `bytes` bytes: one bulk request, or one plain request if it fits a 128-byte line
__device__ __forceinline__ void pf_l2_span(const void* p, uint32_t bytes)
{
    if (bytes <= 128) pf_l2_line(p); else pf_l2_bulk(p, bytes);
}

// twiddles of one butterfly: w^(lo m), m = 1..R-1, from the pass table [m-1][lo].
// Long strides (S >= 64): only w^lo is loaded and the powers are formed by multiplication (depth <= 4, i.e. a few
// ulp, far inside the tolerances): the full table of a long pass ((R-1) S quads, 57 KB for a 4096-point line) does not
// stay in L1 next to the tile and was measured to triple the L2 read traffic of the long-line kernels (C4).
// SPREAD: the lanes of a warp hold (nearly) all different lo -- points-fastest thread order, or fewer than 8 lines per
// tile -- so every table load costs a full 512-byte register writeback: the powers are formed from w^lo for any stride
// >= 8 (measured on the x kernels: -13 % at C3).  With lines-fastest order over >= 8 lines a warp reads 1-4 distinct
// entries per load (cheap broadcasts) and loading stays faster up to stride 32.
template <int LR, int LS, bool SPREAD, typename T>
__device__ __forceinline__ void load_tw(CQ<T>* w, const CQ<T>* __restrict__ tab, int lo)
{
    if (LS >= (SPREAD ? 3 : 6) && LR >= 2) {
        w[1] = ldgq(tab + lo);
        w[2] = cmul(w[1], w[1]); w[3] = cmul(w[2], w[1]);
        if (LR >= 3) { w[4] = cmul(w[2], w[2]); w[5] = cmul(w[4], w[1]); w[6] = cmul(w[3], w[3]); w[7] = cmul(w[4], w[3]); }
        if (LR >= 4) {
            w[8] = cmul(w[4], w[4]);
#pragma unroll
            for (int m = 1; m < 8; ++m) w[8 + m] = cmul(w[8], w[m]);
        }
        return;
    }
#pragma unroll
    for (int m = 1; m < (1 << LR); ++m) w[m] = ldgq(tab + ((m - 1) << LS) + lo);
}
template <int LR, bool INV, typename T>
__device__ __forceinline__ void apply_tw(CQ<T>* a, const CQ<T>* w)
{
#pragma unroll
    for (int m = 1; m < (1 << LR); ++m) a[m] = ctw<INV>(a[m], w[m]);
}

// ---- tile addressing ------------------------------------------------------------------------------------
// A tile parameter PE encodes (pitch, skew) = (PE & 0xffff, PE >> 16): point p of line b sits at
//     s[p * pitch + (p >> 3) * skew + b].
// skew = 0 is the plain point-major tile.  With a skew, threads that walk the butterflies of a stride-1 pass
// (points R i + r, R >= 8) fall into distinct banks even when the tile holds fewer than 8 lines (long lines), and the
// y kernels can run their last forward / first inverse pass butterflies-fastest straight against global memory.
// Strides are multiples of 8, or 1 with radix >= 8, wherever a skewed tile is used, so every leg offset is an immediate.
DM_HDC int tile_pe(int pitch, int skew, bool digit_sum = false) { return pitch + (skew << 16) + (digit_sum ? (1 << 30) : 0); }
// skew term of point p: (p >> 3), or with the digit-sum flag (p >> 3) + (p >> 6) + (p >> 9) + (p >> 12): the bank then
// depends on the SUM of the base-8 digits of p, so positions that differ in any single digit -- in particular the
// digit-reversed positions of consecutive frequencies (the split / merge loops of the x stage) -- never collide.
DM_HDC int tile_skew_term(int PE, int p) { return (PE >> 30) ? (p >> 3) + (p >> 6) + (p >> 9) + (p >> 12) : (p >> 3); }
template <int PE> __device__ __forceinline__ int tile_addr(int p, int b)
{
    constexpr int P = PE & 0xffff, SK = (PE >> 16) & 0x3fff;
    return SK ? p * P + tile_skew_term(PE, p) * SK + b : p * P + b;
}
// offset of leg r (point p0 + r S) from leg 0: p0 has zero bits wherever r S has set bits (in-place passes), so every
// shifted term separates and the offset is a compile-time constant
template <int PE, int S> __host__ __device__ constexpr int tile_leg(int r)
{
    return r * S * (PE & 0xffff) + tile_skew_term(PE, r * S) * ((PE >> 16) & 0x3fff);
}
DM_HDC bool skew_ok(int LL, int POL)      // can a skewed tile be used with this schedule?
{
    const Sched sc = make_sched(LL, POL);
    for (int j = 0; j < sc.n; ++j)
        if (!(sc.ls[j] >= 3 || (sc.ls[j] == 0 && sc.lr[j] >= 3))) return false;
    return true;
}
DM_HDC int tile_quads(int PE, int L, int BL)
{
    return L * (PE & 0xffff) + (((PE >> 16) & 0x3fff) ? tile_skew_term(PE, L) * ((PE >> 16) & 0x3fff) + BL : 0);
}

// ---- one in-place pass over a shared-memory tile, lines fastest ---------------------------------------------
// pass J of schedule SC on lines of length 2^LL; BL lines (quads) per tile; NT threads.
template <typename T, int LL, int POL, int J, bool INV, int BL, int PITCH, int NT>
__device__ __forceinline__ void pass_ss(CQ<T>* s, const CQ<T>* __restrict__ tab, int tid)
{
    constexpr Sched SC = make_sched(LL, POL);
    constexpr int LR = SC.lr[J], LS = SC.ls[J], R = 1 << LR, S = 1 << LS;
    constexpr int NBF = 1 << (LL - LR);            // butterflies per line
    constexpr int TOT = NBF * BL;
    constexpr int ITER = (TOT + NT - 1) / NT;
    constexpr bool HOIST = (LS > 0) && (NT % BL == 0) && ((NT / BL) % S == 0) && ITER > 1;
    constexpr bool SPREAD = BL < 8;
    CQ<T> w[R];
    if (HOIST) load_tw<LR, LS, SPREAD>(w, tab, (tid / BL) & (S - 1));
#pragma unroll(ITER <= 2 ? ITER : 1)
    for (int k = 0; k < ITER; ++k) {
        const int t = tid + k * NT;
        if (TOT % NT != 0 && t >= TOT) break;
        const int b = t % BL, i = t / BL;
        const int lo = i & (S - 1);
        const int p0 = ((i >> LS) << (LS + LR)) + lo;
        CQ<T>* d = s + tile_addr<PITCH>(p0, b);
        CQ<T> a[R];
#pragma unroll
        for (int r = 0; r < R; ++r) a[r] = ldq(d + tile_leg<PITCH, S>(r));
        if (!INV) {
            dftR<LR, false, false>(a);
            if (LS > 0) { if (!HOIST) load_tw<LR, LS, SPREAD>(w, tab, lo); apply_tw<LR, false>(a, w); }
        } else {
            if (LS > 0) { if (!HOIST) load_tw<LR, LS, SPREAD>(w, tab, lo); apply_tw<LR, true>(a, w); }
            dftR<LR, true, false>(a);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) stq(d + tile_leg<PITCH, S>(r), a[r]);
    }
}
// forward passes J..J1-1 (each followed by a barrier) / inverse passes J-1 down to J0
template <typename T, int LL, int POL, int J, int J1, int BL, int PITCH, int NT> struct FwdPasses {
    static __device__ __forceinline__ void run(CQ<T>* s, const TwSet<T>& tw, int tid)
    {
        pass_ss<T, LL, POL, J, false, BL, PITCH, NT>(s, tw.p[J], tid);
        __syncthreads();
        FwdPasses<T, LL, POL, J + 1, J1, BL, PITCH, NT>::run(s, tw, tid);
    }
};
template <typename T, int LL, int POL, int J1, int BL, int PITCH, int NT> struct FwdPasses<T, LL, POL, J1, J1, BL, PITCH, NT> {
    static __device__ __forceinline__ void run(CQ<T>*, const TwSet<T>&, int) {}
};
template <typename T, int LL, int POL, int J0, int J, int BL, int PITCH, int NT> struct InvPasses {   // runs J-1, J-2, .., J0
    static __device__ __forceinline__ void run(CQ<T>* s, const TwSet<T>& tw, int tid)
    {
        pass_ss<T, LL, POL, J - 1, true, BL, PITCH, NT>(s, tw.p[J - 1], tid);
        __syncthreads();
        InvPasses<T, LL, POL, J0, J - 1, BL, PITCH, NT>::run(s, tw, tid);
    }
};
template <typename T, int LL, int POL, int J0, int BL, int PITCH, int NT> struct InvPasses<T, LL, POL, J0, J0, BL, PITCH, NT> {
    static __device__ __forceinline__ void run(CQ<T>*, const TwSet<T>&, int) {}
};

// position of frequency k for schedule (LL, POL), at run time (a few shifts and masks)
template <int LL, int POL> __device__ __forceinline__ int pos_of_freq_rt(int k)
{
    constexpr Sched SC = make_sched(LL, POL);
    int p = 0, w = 0;
#pragma unroll
    for (int j = 0; j < SC.n; ++j) {
        p += ((k >> w) & ((1 << SC.lr[j]) - 1)) << SC.ls[j];
        w += SC.lr[j];
    }
    return p;
}
template <int LL, int POL> __device__ __forceinline__ int freq_of_pos_rt(int p)
{
    constexpr Sched SC = make_sched(LL, POL);
    int k = 0, w = 0;
#pragma unroll
    for (int j = 0; j < SC.n; ++j) {
        k += ((p >> SC.ls[j]) & ((1 << SC.lr[j]) - 1)) << w;
        w += SC.lr[j];
    }
    return k;
}

// first forward pass (pass 0) with the inputs coming from ld(line, point) and the upper half of every line zero
// (the padding); threads walk the point index fastest.  Results go to the tile.
// LF = false: threads walk the point index fastest (lines contiguous in memory); LF = true: lines fastest.
template <typename T, int LL, int POL, int BL, int PITCH, int NT, bool LF, typename LD>
__device__ __forceinline__ void pass_first(CQ<T>* s, const CQ<T>* __restrict__ tab, int tid, LD ld)
{
    constexpr Sched SC = make_sched(LL, POL);
    constexpr int LR = SC.lr[0], LS = SC.ls[0], R = 1 << LR, S = 1 << LS;
    constexpr int TOT = S * BL;
    constexpr int ITER = (TOT + NT - 1) / NT;
    constexpr bool HOIST = (LS > 0) && ITER > 1 && (LF ? (NT % BL == 0 && (NT / BL) % S == 0) : (NT % S == 0));
    constexpr bool SPREAD = !LF || BL < 8;
    CQ<T> w[R];
    if (HOIST) load_tw<LR, LS, SPREAD>(w, tab, LF ? ((tid / BL) & (S - 1)) : (tid & (S - 1)));
    // software pipeline (short loops): the (global) inputs of butterfly k+1 are requested before butterfly k is computed
    constexpr int H = R > 1 ? R / 2 : 1;
    CQ<T> nxt[H];
    auto fetch = [&](int k) {
        const int t = tid + k * NT;
        if (TOT % NT == 0 || t < TOT) {
            const int i = LF ? ((t / BL) & (S - 1)) : (t & (S - 1)), b = LF ? (t % BL) : (t >> LS);
#pragma unroll
            for (int r = 0; r < H; ++r) nxt[r] = ld(b, i + r * S);
        }
    };
    if (ITER <= 4) fetch(0);
#pragma unroll(ITER <= 4 ? ITER : 1)
    for (int k = 0; k < ITER; ++k) {
        const int t = tid + k * NT;
        if (TOT % NT != 0 && t >= TOT) break;
        const int i = LF ? ((t / BL) & (S - 1)) : (t & (S - 1)), b = LF ? (t % BL) : (t >> LS);
        CQ<T> a[R];
        if (ITER > 4) fetch(k);                    // long loops: plain load-use order (fewer live registers)
#pragma unroll
        for (int r = 0; r < H; ++r) a[r] = nxt[r];
        if (ITER <= 4 && k + 1 < ITER) fetch(k + 1);
        dftR<LR, false, true>(a);
        if (LS > 0) { if (!HOIST) load_tw<LR, LS, SPREAD>(w, tab, i); apply_tw<LR, false>(a, w); }
        CQ<T>* d = s + tile_addr<PITCH>(i, b);
#pragma unroll
        for (int r = 0; r < R; ++r) stq(d + tile_leg<PITCH, S>(r), a[r]);
    }
}
// last inverse pass (pass 0 backwards): outputs r < R/2 (the crop) go to st(line, point, value)
template <typename T, int LL, int POL, int BL, int PITCH, int NT, bool LF, typename ST>
__device__ __forceinline__ void pass_last(const CQ<T>* s, const CQ<T>* __restrict__ tab, int tid, ST st)
{
    constexpr Sched SC = make_sched(LL, POL);
    constexpr int LR = SC.lr[0], LS = SC.ls[0], R = 1 << LR, S = 1 << LS;
    constexpr int TOT = S * BL;
    constexpr int ITER = (TOT + NT - 1) / NT;
    constexpr bool HOIST = (LS > 0) && ITER > 1 && (LF ? (NT % BL == 0 && (NT / BL) % S == 0) : (NT % S == 0));
    constexpr bool SPREAD = !LF || BL < 8;
    CQ<T> w[R];
    if (HOIST) load_tw<LR, LS, SPREAD>(w, tab, LF ? ((tid / BL) & (S - 1)) : (tid & (S - 1)));
#pragma unroll(ITER <= 2 ? ITER : 1)
    for (int k = 0; k < ITER; ++k) {
        const int t = tid + k * NT;
        if (TOT % NT != 0 && t >= TOT) break;
        const int i = LF ? ((t / BL) & (S - 1)) : (t & (S - 1)), b = LF ? (t % BL) : (t >> LS);
        const CQ<T>* d = s + tile_addr<PITCH>(i, b);
        CQ<T> a[R];
#pragma unroll
        for (int r = 0; r < R; ++r) a[r] = ldq(d + tile_leg<PITCH, S>(r));
        if (LS > 0) { if (!HOIST) load_tw<LR, LS, SPREAD>(w, tab, i); apply_tw<LR, true>(a, w); }
        dftR<LR, true, false>(a);
#pragma unroll
        for (int r = 0; r < R / 2; ++r) st(b, i + r * S, a[r]);
    }
}

// =========================================================================================== K2v / K4v: y stage
// lines l = (c*nq + ql)*nz + z of the slab [q0, q0+nq); a tile = BP consecutive lines (quads: two x-frequencies each).
__device__ __forceinline__ long long w1v_line_offset(const GeoV& g, int l, int q0, int nq)
{
    const int z = l % g.nz, ck = l / g.nz, ql = ck % nq, c = ck / nq;
    return (((long long)c * g.hq + q0 + ql) * g.nz + z) * g.ny;
}

// W2v order of a y line ("position order"): with NP >= 2 passes the last forward pass (stride 1, radix R, butterfly i
// = points R i .. R i + R - 1) stores its output r of butterfly i at  r * (Ny / R) + i  -- consecutive threads write
// consecutive quads, straight from registers -- and the first inverse pass loads the same way.  The stored kernel
// spectrum follows the same order (ypos2freq, v2_host.cuh: y_w2_pos_to_tile_pos).
// y forward FFT, zero padding synthesised (PAPER.md:309-315 yFFT): W1v -> W2v
template <typename T, int LNY, int POL, int BP, int NT>
__global__ void __launch_bounds__(NT, (POL == 6 && NT <= 128 ? 3 : 0)) k_y_fwd_v(GeoV g, int q0, int nq, const CQ<T>* __restrict__ W1,
                                               CQ<T>* __restrict__ W2, TwSet<T> tw)
{
    pdl_enter(g);
    constexpr Sched SC = make_sched(LNY, POL);
    constexpr int NP = SC.n;
    constexpr int NY = 1 << LNY, PITCH = tile_pe(BP | 1, NP >= 2 ? 1 : 0, POL == 6);
    CQ<T>* s = reinterpret_cast<CQ<T>*>(smem_v2);
    __shared__ long long loff[BP];
    const int tid = threadIdx.x;
    const int nlines = 3 * nq * g.nz;
    const int l0 = blockIdx.x * BP;
    if (tid < BP) loff[tid] = (l0 + tid < nlines) ? w1v_line_offset(g, l0 + tid, q0, nq) : -1;
    if (g.pf && tid < BP) {
        const long long lp = (long long)(blockIdx.x + g.pf) * BP + tid;
        if (lp < nlines) pf_l2_bulk(W1 + w1v_line_offset(g, (int)lp, q0, nq), (uint32_t)(g.ny * sizeof(CQ<T>)));
    }
    __syncthreads();
    auto ld = [&](int b, int p) { const long long o = loff[b]; return o >= 0 ? ldsq(W1 + o + p) : cq_zero<T>(); };
    pass_first<T, LNY, POL, BP, PITCH, NT, false>(s, tw.p[0], tid, ld);
    __syncthreads();
    CQ<T>* dst = W2 + (size_t)l0 * NY;
    const int nvalid = min(BP, nlines - l0);
    if constexpr (NP >= 2) {
        FwdPasses<T, LNY, POL, 1, NP - 1, BP, PITCH, NT>::run(s, tw, tid);
        // last pass (stride 1, no twiddles): butterflies fastest, results straight to global
        constexpr int LR = SC.lr[NP - 1], R = 1 << LR, LNB = LNY - LR, NBF = 1 << LNB, TOT = NBF * BP;
        static_assert(SC.ls[NP - 1] == 0 && R >= 8, "last pass: stride 1, radix >= 8");
#pragma unroll(R >= 32 ? 1 : 2)
        for (int t = tid; t < TOT; t += NT) {
            const int i = t & (NBF - 1), b = t >> LNB;
            const CQ<T>* d = s + tile_addr<PITCH>(i << LR, b);
            CQ<T> a[R];
#pragma unroll
            for (int r = 0; r < R; ++r) a[r] = ldq(d + tile_leg<PITCH, 1>(r));
            dftR<LR, false, false>(a);
            if (b < nvalid) {
#pragma unroll
                for (int r = 0; r < R; ++r) stq(dst + ((size_t)b << LNY) + (r << LNB) + i, a[r]);
            }
        }
    } else {
#pragma unroll 4
        for (int idx = tid; idx < (nvalid << LNY); idx += NT) {
            const int b = idx >> LNY, p = idx & (NY - 1);
            stq(dst + idx, ldq(s + tile_addr<PITCH>(p, b)));
        }
    }
}

// Long lines (one line pair per tile: Ny >= 4096): persistent blocks, one per SM.  The zero-padded input half of the
// NEXT line is bulk-copied (cp.async.bulk + mbarrier) into a staging buffer while the current line is transformed, so
// the block never waits for its input (with a single resident block nothing else hides that latency).
template <typename T, int LNY, int POL, int NT>
__global__ void __launch_bounds__(NT) k_y_fwd_long_v(GeoV g, int q0, int nq, const CQ<T>* __restrict__ W1,
                                                    CQ<T>* __restrict__ W2, TwSet<T> tw)
{
    pdl_enter(g);
    constexpr Sched SC = make_sched(LNY, POL);
    constexpr int NP = SC.n;
    static_assert(NP >= 2, "long lines have several passes");
    constexpr int NY = 1 << LNY, PITCH = tile_pe(1, 1, POL == 6), TQ = tile_quads(PITCH, NY, 1);
    constexpr uint32_t kBytes = (uint32_t)((NY / 2) * sizeof(CQ<T>));
    CQ<T>* s = reinterpret_cast<CQ<T>*>(smem_v2);
    CQ<T>* stage = s + TQ;
    __shared__ uint64_t mbar;
    const int tid = threadIdx.x;
    const int nlines = 3 * nq * g.nz;
    if (tid == 0) { mbar_init(&mbar, 1); fence_mbar_init(); }
    __syncthreads();
    int line = blockIdx.x;
    if (tid == 0 && line < nlines) { mbar_arrive_expect_tx(&mbar, kBytes); bulk_g2s(stage, W1 + w1v_line_offset(g, line, q0, nq), kBytes, &mbar); }
    for (int it = 0; line < nlines; line += gridDim.x, ++it) {
        mbar_wait(&mbar, (uint32_t)(it & 1));
        auto ld = [&](int, int p) { return ldq(stage + p); };
        pass_first<T, LNY, POL, 1, PITCH, NT, false>(s, tw.p[0], tid, ld);
        __syncthreads();                                       // staging buffer consumed, tile written
        const int next = line + gridDim.x;
        if (tid == 0 && next < nlines) { mbar_arrive_expect_tx(&mbar, kBytes); bulk_g2s(stage, W1 + w1v_line_offset(g, next, q0, nq), kBytes, &mbar); }
        FwdPasses<T, LNY, POL, 1, NP - 1, 1, PITCH, NT>::run(s, tw, tid);
        constexpr int LR = SC.lr[NP - 1], R = 1 << LR, LNB = LNY - LR, NBF = 1 << LNB;
        CQ<T>* dst = W2 + (size_t)line * NY;
#pragma unroll(R >= 32 ? 1 : 2)
        for (int i = tid; i < NBF; i += NT) {
            const CQ<T>* d = s + tile_addr<PITCH>(i << LR, 0);
            CQ<T> a[R];
#pragma unroll
            for (int r = 0; r < R; ++r) a[r] = ldq(d + tile_leg<PITCH, 1>(r));
            dftR<LR, false, false>(a);
#pragma unroll
            for (int r = 0; r < R; ++r) stq(dst + (r << LNB) + i, a[r]);
        }
        __syncthreads();                                       // tile free for the next line
    }
}

// y inverse FFT fused with the crop: W2v -> W1v
template <typename T, int LNY, int POL, int BP, int NT, bool SH>
__device__ __forceinline__ void y_inv_body(const GeoV& g, int q0, int nq, const CQ<T>* __restrict__ W2,
                                           CQ<T>* __restrict__ W1, const ShardMap<T>* map, const TwSet<T>& tw)
{
    constexpr Sched SC = make_sched(LNY, POL);
    constexpr int NP = SC.n;
    constexpr int NY = 1 << LNY, PITCH = tile_pe(BP | 1, NP >= 2 ? 1 : 0, POL == 6);
    CQ<T>* s = reinterpret_cast<CQ<T>*>(smem_v2);
    __shared__ long long loff[BP];
    const int tid = threadIdx.x;
    const int nlines = 3 * nq * g.nz;
    const int l0 = blockIdx.x * BP;
    if (tid < BP) {
        long long o = -1;
        if (l0 + tid < nlines) {
            if constexpr (SH) {      // global line number ((c hq + q) nz + z) of the partitioned W1out
                const int l = l0 + tid, z = l % g.nz, ck = l / g.nz, ql = ck % nq, c = ck / nq;
                o = ((long long)c * map->pitch + map->off + q0 + ql) * g.nz + z;
            } else o = w1v_line_offset(g, l0 + tid, q0, nq);
        }
        loff[tid] = o;
    }
    const CQ<T>* src = W2 + (size_t)l0 * NY;
    const int nvalid = min(BP, nlines - l0);
    if (g.pf && tid < BP) {
        const long long lp = (long long)(blockIdx.x + g.pf) * BP + tid;
        if (lp < nlines) pf_l2_bulk(W2 + (size_t)lp * NY, (uint32_t)(NY * sizeof(CQ<T>)));
    }
    if constexpr (NP >= 2) {
        // first inverse pass (stride 1, no twiddles): inputs straight from global, butterflies fastest
        constexpr int LR = SC.lr[NP - 1], R = 1 << LR, LNB = LNY - LR, NBF = 1 << LNB, TOT = NBF * BP;
#pragma unroll(R >= 32 ? 1 : 2)
        for (int t = tid; t < TOT; t += NT) {
            const int i = t & (NBF - 1), b = t >> LNB;
            CQ<T> a[R];
#pragma unroll
            for (int r = 0; r < R; ++r) a[r] = b < nvalid ? ldsq(src + ((size_t)b << LNY) + (r << LNB) + i) : cq_zero<T>();
            dftR<LR, true, false>(a);
            CQ<T>* d = s + tile_addr<PITCH>(i << LR, b);
#pragma unroll
            for (int r = 0; r < R; ++r) stq(d + tile_leg<PITCH, 1>(r), a[r]);
        }
        __syncthreads();
        InvPasses<T, LNY, POL, 1, NP - 1, BP, PITCH, NT>::run(s, tw, tid);
    } else {
#pragma unroll 4
        for (int idx = tid; idx < (BP << LNY); idx += NT) {
            const int b = idx >> LNY, p = idx & (NY - 1);
            stq(s + tile_addr<PITCH>(p, b), b < nvalid ? ldsq(src + idx) : cq_zero<T>());
        }
        __syncthreads();
    }
    if constexpr (SH) {
        // row y of line L belongs to rank r = y / per: its W1out holds [line][ny_r] (Transfer_S2_to_S1)
        auto st = [&](int b, int p, CQ<T> v) {
            const long long o = loff[b];
            if (o < 0) return;
            const int r = min(p / map->per, map->G - 1), y0 = r * map->per;
            const int nyr = r == map->G - 1 ? map->total - y0 : map->per;
            stq(map->base[r] + o * nyr + (p - y0), v);
        };
        pass_last<T, LNY, POL, BP, PITCH, NT, false>(s, tw.p[0], tid, st);
    } else {
        auto st = [&](int b, int p, CQ<T> v) { const long long o = loff[b]; if (o >= 0) stq(W1 + o + p, v); };
        pass_last<T, LNY, POL, BP, PITCH, NT, false>(s, tw.p[0], tid, st);
    }
}
template <typename T, int LNY, int POL, int BP, int NT>
__global__ void __launch_bounds__(NT, (POL == 6 && NT <= 128 ? 3 : 0)) k_y_inv_v(GeoV g, int q0, int nq, const CQ<T>* __restrict__ W2,
                                               CQ<T>* __restrict__ W1, TwSet<T> tw)
{
    pdl_enter(g);
    y_inv_body<T, LNY, POL, BP, NT, false>(g, q0, nq, W2, W1, nullptr, tw);
    pdl_leave(g);
}
// the same with the crop scattered to the ranks that own the rows (several GPUs)
template <typename T, int LNY, int POL, int BP, int NT>
__global__ void __launch_bounds__(NT) k_y_inv_sh_v(GeoV g, int q0, int nq, const CQ<T>* __restrict__ W2,
                                                  const __grid_constant__ ShardMap<T> map, TwSet<T> tw)
{
    pdl_enter(g);
    y_inv_body<T, LNY, POL, BP, NT, true>(g, q0, nq, W2, nullptr, &map, tw);
    pdl_leave(g);
}

// =========================================================================================== K3v: z stage
// z FFT . kernel multiplication . z IFFT "in the same routine" (PAPER.md:343; :316-326 zFFT, KernelMultiplication).
// One (q, kz', py) entry is NCH chunks of 16 bytes, chunk j of column ty at p[j * KT]:
// fp32: 3 chunks {xx0,xx1,yy0,yy1} {zz0,zz1,xy0,xy1} {xz0,xz1,yz0,yz1};  fp64: 6 chunks, one component pair each.
template <typename T> struct kchunks;
template <> struct kchunks<float>  { static constexpr int N = 3; using V = float4; };
template <> struct kchunks<double> { static constexpr int N = 6; using V = double2; };
template <int KT> __device__ __forceinline__ KQ<float> ldk(const float4* p)
{
    const float4 a = __ldg(p), b = __ldg(p + KT), c = __ldg(p + 2 * KT);
    KQ<float> k;
    k.xx = make_float2(a.x, a.y); k.yy = make_float2(a.z, a.w); k.zz = make_float2(b.x, b.y);
    k.xy = make_float2(b.z, b.w); k.xz = make_float2(c.x, c.y); k.yz = make_float2(c.z, c.w);
    return k;
}
template <int KT> __device__ __forceinline__ KQ<double> ldk(const double2* p)
{
    KQ<double> k;
    k.xx = __ldg(p); k.yy = __ldg(p + KT); k.zz = __ldg(p + 2 * KT); k.xy = __ldg(p + 3 * KT); k.xz = __ldg(p + 4 * KT); k.yz = __ldg(p + 5 * KT);
    return k;
}
// H^_a = sum_b K^_ab M^_b, K^ real and symmetric.  SGN: sign of the z-odd components xz, yz
// (+1 direct, -1 mirrored kz > Nz/2, 0 = run-time sign sg).  sy: sign of the y-odd components xy, yz (-1 for a
// column whose y frequency is mirrored, yslot < 0).  FILM (the routine run along y): sy = 1, the stored slots are permuted.
template <int SGN, typename T>
__device__ __forceinline__ void apply_kernel(const KQ<T>& k, CQ<T>& mx, CQ<T>& my, CQ<T>& mz, T sg, T sy)
{
    typename vec2<T>::type kxz = k.xz, kyz = vmul(k.yz, vdup(sy));
    const typename vec2<T>::type kxy = vmul(k.xy, vdup(sy));
    if (SGN < 0) { kxz = vneg(kxz); kyz = vneg(kyz); }
    if (SGN == 0) { kxz = vmul(kxz, vdup(sg)); kyz = vmul(kyz, vdup(sg)); }
    CQ<T> hx, hy, hz;
    hx.re = vfma(kxz, mz.re, vfma(kxy, my.re, vmul(k.xx, mx.re)));
    hx.im = vfma(kxz, mz.im, vfma(kxy, my.im, vmul(k.xx, mx.im)));
    hy.re = vfma(kyz, mz.re, vfma(k.yy, my.re, vmul(kxy, mx.re)));
    hy.im = vfma(kyz, mz.im, vfma(k.yy, my.im, vmul(kxy, mx.im)));
    hz.re = vfma(k.zz, mz.re, vfma(kyz, my.re, vmul(kxz, mx.re)));
    hz.im = vfma(k.zz, mz.im, vfma(kyz, my.im, vmul(kxz, mx.im)));
    mx = hx; my = hy; mz = hz;
}

// multiply the RF points of one fused butterfly (positions p0..p0+RF-1 <-> kz = f0 + m Nz/RF); Kcol = this column's
// first chunk at kz' = 0, rows kz' are kchunks<T>::N * KT vectors apart
template <typename T, int LNZ, int LRF, int KT, int M> struct MulPoints {
    using KV = typename kchunks<T>::V;
    static __device__ __forceinline__ void run(CQ<T> (*a)[1 << LRF], const KV* __restrict__ Kcol, int f0, T sy)
    {
        constexpr int NZ = 1 << LNZ, RF = 1 << LRF, W = NZ >> LRF, ROW = kchunks<T>::N * KT;
        const int kz = f0 + M * W;
        if (RF == 1 || 2 * M < RF) {
            apply_kernel<1>(ldk<KT>(Kcol + kz * ROW), a[0][M], a[1][M], a[2][M], (T)1, sy);
        } else if (2 * M > RF) {
            apply_kernel<-1>(ldk<KT>(Kcol + (NZ - kz) * ROW), a[0][M], a[1][M], a[2][M], (T)1, sy);
        } else {
            const bool mir = f0 > 0;
            apply_kernel<0>(ldk<KT>(Kcol + (mir ? NZ - kz : kz) * ROW), a[0][M], a[1][M], a[2][M], mir ? (T)-1 : (T)1, sy);
        }
        MulPoints<T, LNZ, LRF, KT, M + 1>::run(a, Kcol, f0, sy);
    }
};
template <typename T, int LNZ, int LRF, int KT> struct MulPoints<T, LNZ, LRF, KT, (1 << LRF)> {
    using KV = typename kchunks<T>::V;
    static __device__ __forceinline__ void run(CQ<T> (*)[1 << LRF], const KV* __restrict__, int, T) {}
};
// slot and y sign of W2v position py (yslot == nullptr: one-cell-thick mesh, the routine runs along y: slot 0)
// -> offset (in 16-byte vectors) of the column's first chunk at kz' = 0 inside the pair plane of the stored spectrum
template <int KT, int NCH> __device__ __forceinline__ size_t kslot(const int* __restrict__ yslot, int py, int kpz, float& sy)
{
    if (!yslot) { sy = 1.f; return 0; }
    const int v = __ldg(yslot + py);
    sy = v < 0 ? -1.f : 1.f;
    const int slot = v & 0x7fffffff;
    return (size_t)(slot / KT) * kpz * (NCH * KT) + slot % KT;
}

// Nz >= 16 (at least two passes).  Tile = one pair plane ql x TY consecutive py x all z x 3 components:
// shared s[Nz][3 TY] quads, lines fastest everywhere (a warp's accesses are consecutive quads: conflict free).
//
// FILM = true (TY == 1): the same routine run along y on the x-stage workspace of a one-cell-thick mesh
// (scope row a3': y FFT . multiply . y IFFT in one kernel, in place on W1v[3][hq][ny]; call it with g.nz = ny,
// g.Nz = Ny, g.Ny = 1, nq = hq).  The transform axis is y, so the components that change sign on a mirrored
// frequency are xy and yz: the three lines are taken in the order (x, z, y) and the stored spectrum is permuted
// to match at plan time (k_pack_film_v), which turns "odd in z" into "odd in y" without touching this code.
template <typename T, int LNZ, int POL, int TY, int NT, int MINB, bool FILM = false>
__global__ void __launch_bounds__(NT, MINB) k_z_v(GeoV g, int q0, int nq, CQ<T>* W2, const typename kchunks<T>::V* __restrict__ K,
                                                  const int* __restrict__ yslot, TwSet<T> tw, const __grid_constant__ CUtensorMap tmap)
{
    pdl_enter(g);
    constexpr int NZ = 1 << LNZ, B = 3 * TY;
    constexpr Sched SC = make_sched(LNZ, POL);
    constexpr int NP = SC.n, LRF = SC.lr[NP - 1], RF = 1 << LRF;
    static_assert(NP >= 2 && NT % TY == 0 && (!FILM || TY == 1), "k_z_v: needs >= 2 passes");
    constexpr int PE = tile_pe(B, (TY <= 2 && skew_ok(LNZ, POL)) ? TY : 0);     // narrow tiles: skewed (bank conflicts)
    CQ<T>* s = reinterpret_cast<CQ<T>*>(smem_v2);
    const int tid = threadIdx.x;
    const int tilesY = g.Ny / TY;
    const int pyt = blockIdx.x % tilesY, ql = blockIdx.x / tilesY;
    const int py0 = pyt * TY;
    const size_t cstride = (size_t)nq * g.nz * g.Ny;
    CQ<T>* base = W2 + (size_t)ql * g.nz * g.Ny + py0;
    const int Ny = g.Ny;
    if (g.pf && blockIdx.x + g.pf < gridDim.x) {
        const int bn = blockIdx.x + g.pf, pytn = bn % tilesY, qln = bn / tilesY;
        const CQ<T>* bnx = W2 + (size_t)qln * g.nz * g.Ny + pytn * TY;
        if (FILM) { if (tid < 3) pf_l2_bulk(bnx + tid * cstride, (uint32_t)(g.nz * sizeof(CQ<T>))); }
        else if (g.pft) { if (tid == 0) pf_l2_tensor(&tmap, pytn * TY * 4, 0, qln, 0); }       // box {TY quads, nz, 1 pair plane, 3 components}
        else for (int r = tid; r < 3 * g.nz; r += NT) { const int c = r / g.nz, z = r - c * g.nz; pf_l2_span(bnx + c * cstride + (size_t)z * Ny, (uint32_t)(TY * sizeof(CQ<T>))); }
        if (!FILM && tid >= NT - 2) {
            // the spectrum rows of that tile: the slot tile(s) its first and last column fall into (contiguous kpz rows each)
            const int sl = __ldg(yslot + pytn * TY + (tid == NT - 1 ? TY - 1 : 0)) & 0x7fffffff;
            const uint32_t kb = (uint32_t)(g.kpz * kchunks<T>::N * TY * sizeof(typename kchunks<T>::V));
            pf_l2_bulk(K + ((size_t)(q0 + qln) * g.kst + sl / TY) * g.kpz * (kchunks<T>::N * TY), kb);
        }
    }
    // this thread's column in the fused pass (NT % TY == 0: the same for every item) and its slot in the stored spectrum
    float sy;
    const size_t slot = kslot<TY, kchunks<T>::N>(yslot, py0 + tid % TY, g.kpz, sy);
    auto ld = [&](int b, int z) { const int c = FILM ? (b == 0 ? 0 : 3 - b) : b / TY, ty = FILM ? 0 : b - c * TY; return ldsq(base + c * cstride + (size_t)z * Ny + ty); };
    pass_first<T, LNZ, POL, B, PE, NT, true>(s, tw.p[0], tid, ld);
    __syncthreads();
    FwdPasses<T, LNZ, POL, 1, NP - 1, B, PE, NT>::run(s, tw, tid);
    const typename kchunks<T>::V* Kq = K + (size_t)(q0 + ql) * g.kst * g.kpz * (kchunks<T>::N * TY);   // KT == TY
    auto load_fwd = [&](CQ<T> (*a)[RF], int p0, int ty) {
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) {
#pragma unroll
            for (int m = 0; m < RF; ++m) a[cc][m] = ldq(s + tile_addr<PE>(p0, cc * TY + ty) + tile_leg<PE, 1>(m));
            dftR<LRF, false, false>(a[cc]);
        }
    };
    auto inv_store = [&](CQ<T> (*a)[RF], int p0, int ty) {
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) {
            dftR<LRF, true, false>(a[cc]);
#pragma unroll
            for (int m = 0; m < RF; ++m) stq(s + tile_addr<PE>(p0, cc * TY + ty) + tile_leg<PE, 1>(m), a[cc][m]);
        }
    };
    if constexpr (LRF == 3 && sizeof(T) == 4 && ((NZ >> 4) * TY >= NT)) {      // (enough pairs to occupy every thread)
        // fused: last forward pass . multiply . first inverse pass, TWO butterflies per work unit.  Butterfly f (0 <= f < W,
        // W = Nz / 8) holds kz = f + m W, m = 0..7; its points m >= 4 are mirrored frequencies whose packed rows
        // Nz - kz = (W - f) + (7 - m) W are the DIRECT rows of butterfly W - f, and vice versa: the pair (f, W - f) shares
        // its eight spectrum rows, which are loaded once (they were loaded twice when every butterfly fetched its own:
        // 1/8 of the z stage's L1 wavefronts).  Unit 0 is the self-mirrored pair (0, W/2): same code, a select picks its
        // rows (butterfly 0: rows 0, W, .., 4W, 3W, .., W; butterfly W/2: its own four rows both ways).
        constexpr int W = NZ >> 3, UNITS = (W / 2) * TY, ITER = (UNITS + NT - 1) / NT, ROW = kchunks<T>::N * TY;
        const typename kchunks<T>::V* Kcol = Kq + slot;
#pragma unroll 1
        for (int k = 0; k < ITER; ++k) {
            const int t = tid + k * NT;
            if (UNITS % NT != 0 && t >= UNITS) break;
            const int ty = t % TY, u = t / TY;
            const bool self = u == 0;
            const int fA = u, fB = self ? W / 2 : W - u;
            KQ<T> KA[4], KB[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) { KA[j] = ldk<TY>(Kcol + (fA + j * W) * ROW); KB[j] = ldk<TY>(Kcol + (fB + j * W) * ROW); }
            const KQ<T> KN = ldk<TY>(Kcol + (self ? 4 * W : fB + 3 * W) * ROW);      // row Nz/2 (unit 0 only; else KB[3] again: a hit)
            auto ksel = [](bool c, const KQ<T>& x, const KQ<T>& y) {
                KQ<T> r;
                r.xx = c ? x.xx : y.xx; r.yy = c ? x.yy : y.yy; r.zz = c ? x.zz : y.zz; r.xy = c ? x.xy : y.xy; r.xz = c ? x.xz : y.xz; r.yz = c ? x.yz : y.yz;
                return r;
            };
            CQ<T> a[3][RF];
            {   // butterfly A
                const int p0 = pos_of_freq_rt<LNZ, POL>(fA);
                load_fwd(a, p0, ty);
#pragma unroll
                for (int m = 0; m < 4; ++m) apply_kernel<1>(KA[m], a[0][m], a[1][m], a[2][m], (T)1, (T)sy);
                apply_kernel<0>(ksel(self, KN, KB[3]), a[0][4], a[1][4], a[2][4], self ? (T)1 : (T)-1, (T)sy);
#pragma unroll
                for (int m = 5; m < 8; ++m) apply_kernel<-1>(ksel(self, KA[8 - m], KB[7 - m]), a[0][m], a[1][m], a[2][m], (T)1, (T)sy);
                inv_store(a, p0, ty);
            }
            {   // butterfly B
                const int p0 = pos_of_freq_rt<LNZ, POL>(fB);
                load_fwd(a, p0, ty);
#pragma unroll
                for (int m = 0; m < 4; ++m) apply_kernel<1>(KB[m], a[0][m], a[1][m], a[2][m], (T)1, (T)sy);
#pragma unroll
                for (int m = 4; m < 8; ++m) apply_kernel<-1>(ksel(self, KB[7 - m], KA[7 - m]), a[0][m], a[1][m], a[2][m], (T)1, (T)sy);
                inv_store(a, p0, ty);
            }
        }
    } else {   // fused: last forward pass . multiply . first inverse pass; item = (butterfly i, column ty), 3 components
        constexpr int NBF = NZ >> LRF, TOT = NBF * TY, ITER = (TOT + NT - 1) / NT;
#pragma unroll 1
        for (int k = 0; k < ITER; ++k) {
            const int t = tid + k * NT;
            if (TOT % NT != 0 && t >= TOT) break;
            const int ty = t % TY, i = t / TY;
            const int p0 = i << LRF;
            CQ<T> a[3][RF];
            load_fwd(a, p0, ty);
            const int f0 = freq_of_pos_rt<LNZ, POL>(p0);
            MulPoints<T, LNZ, LRF, TY, 0>::run(a, Kq + slot, f0, (T)sy);
            inv_store(a, p0, ty);
        }
    }
    __syncthreads();
    InvPasses<T, LNZ, POL, 1, NP - 1, B, PE, NT>::run(s, tw, tid);
    auto st = [&](int b, int z, CQ<T> v) { const int c = FILM ? (b == 0 ? 0 : 3 - b) : b / TY, ty = FILM ? 0 : b - c * TY; stq(base + c * cstride + (size_t)z * Ny + ty, v); };
    pass_last<T, LNZ, POL, B, PE, NT, true>(s, tw.p[0], tid, st);
    pdl_leave(g);
}

// Nz <= 8: the whole z transform of a column is one butterfly per component in registers; no shared memory.
// grid = nq * Ny / 128 (or fewer columns per block if Ny < 128), block = min(Ny, 128).
template <typename T, int LNZ>
__global__ void __launch_bounds__(128) k_z1_v(GeoV g, int q0, int nq, CQ<T>* W2, const typename kchunks<T>::V* __restrict__ K,
                                              const int* __restrict__ yslot)
{
    pdl_enter(g);
    constexpr int RF = 1 << LNZ;
    const int cols = blockDim.x;
    const int tilesY = g.Ny / cols;
    const int pyt = blockIdx.x % tilesY, ql = blockIdx.x / tilesY;
    const int py = pyt * cols + threadIdx.x;
    const size_t cstride = (size_t)nq * g.nz * g.Ny;
    CQ<T>* col = W2 + (size_t)ql * g.nz * g.Ny + py;
    const int Ny = g.Ny;
    CQ<T> a[3][RF];
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) {
#pragma unroll
        for (int m = 0; m < (RF > 1 ? RF / 2 : 1); ++m) a[cc][m] = ldq(col + cc * cstride + (size_t)m * Ny);
        dftR<LNZ, false, true>(a[cc]);
    }
    float sy;
    const size_t slot = kslot<32, kchunks<T>::N>(yslot, py, g.kpz, sy);                                  // KT = 32
    MulPoints<T, LNZ, LNZ, 32, 0>::run(a, K + (size_t)(q0 + ql) * g.kst * g.kpz * (kchunks<T>::N * 32) + slot, 0, (T)sy);
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) {
        dftR<LNZ, true, false>(a[cc]);
#pragma unroll
        for (int m = 0; m < (RF > 1 ? RF / 2 : 1); ++m) stq(col + cc * cstride + (size_t)m * Ny, a[cc][m]);
    }
}

// Nz = 16 (8 cells thick: C4), fp32: the whole z stage of a column in the registers of TWO lanes, no shared memory.
// The 16-point transform of [8 values, 8 zeros] splits by frequency parity into two 8-point transforms of the same
// 8 values (decimation in frequency with a zero upper half):
//     M^[2k]   = DFT8(m[z])[k]                      lane "E"  (kz = 0, 2, .., 14)
//     M^[2k-1] = DFT8(m[z] conj(w16^z))[k]          lane "O"  (kz = 15, 1, 3, .., 13)
// and the kept half of the inverse is the sum of the two lanes' 8-point inverses,
//     h[z] = IDFT8(H^e)[z] + w16^z IDFT8(H^o)[z],   z = 0..7,
// exchanged with one shuffle per value (lane ^ 16).  Lanes 0-15 / 16-31 of a warp are the E / O halves of the same 16
// columns, so their loads coalesce to the same sectors.  Each thread has 24 + 24 independent 128-bit loads in flight
// (field + kernel spectrum): the latency is covered without shared-memory staging, and the stage moves one
// shared-memory-free wavefront per 128 bytes.  grid = nq * Ny / 64, block = 128.
template <typename T, int MINB>
__global__ void __launch_bounds__(128, MINB) k_z16_v(GeoV g, int q0, int nq, CQ<T>* W2, const typename kchunks<T>::V* __restrict__ K,
                                                  const int* __restrict__ yslot)
{
    pdl_enter(g);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const bool odd = (lane >> 4) != 0;
    const int tilesY = g.Ny >> 6;
    const int pyt = blockIdx.x % tilesY, ql = blockIdx.x / tilesY;
    const int py = (pyt << 6) + (wid << 4) + (lane & 15);
    const int Ny = g.Ny;
    const size_t cstride = (size_t)nq * 8 * Ny;
    CQ<T>* col = W2 + (size_t)ql * 8 * Ny + py;
    CQ<T> a[3][8];
#pragma unroll
    for (int cc = 0; cc < 3; ++cc)
#pragma unroll
        for (int z = 0; z < 8; ++z) a[cc][z] = ldsq(col + cc * cstride + (size_t)z * Ny);
    // w16^z of the O lanes (1 on the E lanes)
    const T c8 = (T)0.92387953251128675613, s8 = (T)0.38268343236508977173, h8 = (T)0.70710678118654752440;
    const T wr[8] = {(T)1, c8, h8, s8, (T)0, -s8, -h8, -c8}, wi[8] = {(T)0, -s8, -h8, -c8, (T)-1, -c8, -h8, -s8};
    CQ<T> tw[8];
#pragma unroll
    for (int z = 1; z < 8; ++z) { tw[z].re = vdup(odd ? wr[z] : (T)1); tw[z].im = vdup(odd ? wi[z] : (T)0); }
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) {
#pragma unroll
        for (int z = 1; z < 8; ++z) a[cc][z] = cmulc(a[cc][z], tw[z]);
        dft8<false, false>(a[cc]);
    }
    // point k of the lane is kz = 2k (E) or 2k-1 mod 16 (O); rows of the z-packed spectrum and the sign of its z-odd
    // components (mirrored frequencies kz > 8):   E: 0 2 4 6 8 6 4 2 / + + + + + - - -    O: 1 1 3 5 7 7 5 3 / - + + + + - - -
    float sy;
    const size_t slot = kslot<32, kchunks<T>::N>(yslot, py, 9, sy);                                      // KT = 32
    constexpr int ROW = kchunks<T>::N * 32;
    const typename kchunks<T>::V* Kc = K + (size_t)(q0 + ql) * g.kst * 9 * ROW + slot;
    if (g.pf) {   // the spectrum rows are consumed late (registers): ask for them now
#pragma unroll
        for (int k = 0; k < 5; ++k)
#pragma unroll
            for (int j = 0; j < kchunks<T>::N; ++j) pf_l2_line(Kc + (2 * k + (odd ? 1 : 0) - (odd && k == 4 ? 2 : 0)) * ROW + j * 32);
    }
    constexpr int rowE[8] = {0, 2, 4, 6, 8, 6, 4, 2}, rowO[8] = {1, 1, 3, 5, 7, 7, 5, 3};
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int row = odd ? rowO[k] : rowE[k];
        const T sg = (k >= 5 || (k == 0 && odd)) ? (T)-1 : (T)1;
        apply_kernel<0>(ldk<32>(Kc + row * ROW), a[0][k], a[1][k], a[2][k], sg, (T)sy);
    }
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) {
        dft8<true, false>(a[cc]);
#pragma unroll
        for (int z = 1; z < 8; ++z) a[cc][z] = cmul(a[cc][z], tw[z]);
    }
    // h[z] = E part + O part: the E lane finishes z = 0..3, the O lane z = 4..7
#pragma unroll
    for (int cc = 0; cc < 3; ++cc)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const CQ<T> give = odd ? a[cc][j] : a[cc][j + 4], keep = odd ? a[cc][j + 4] : a[cc][j];
            CQ<T> got;
            got.re.x = __shfl_xor_sync(0xffffffffu, give.re.x, 16); got.re.y = __shfl_xor_sync(0xffffffffu, give.re.y, 16);
            got.im.x = __shfl_xor_sync(0xffffffffu, give.im.x, 16); got.im.y = __shfl_xor_sync(0xffffffffu, give.im.y, 16);
            stq(col + cc * cstride + (size_t)(j + (odd ? 4 : 0)) * Ny, cadd(keep, got));
        }
    pdl_leave(g);
}

// Nz = 256 / 512 (fp32): the zero-padded z transform as TWO independent half-length transforms of the same nz inputs
// (decimation in frequency with a zero upper half, as in k_z16_v):
//     M^[2k]   = DFT_{Nz/2}(m[z])[k]                 "E" tile,   M^[2k+1] = DFT_{Nz/2}(m[z] w_Nz^z)[k]      "O" tile,
// and the cropped inverse  h[z] = IDFT_{Nz/2}(H^_even)[z] + conj(w_Nz^z) IDFT_{Nz/2}(H^_odd)[z],  z < nz.
// A half-length transform is TWO passes, radix Nz/16 (16 or 32, straight from / to global memory, in registers) and
// radix 8 (the fused pass: last forward . multiply . first inverse), where the padded length needs three (4.8.8 / 8.8.8):
// every point of the tile is written and read twice instead of four times.  The shared-memory traffic is what bounds the
// z stage of long columns (C5: 68 % of the L1 data pipe with the three-pass kernel).
// Lanes 0-15 / 16-31 of a warp are the E / O halves of the same 16 (butterfly, line) items: they load the same addresses
// and exchange their halves of the inverse by one shuffle per value.  The fused pass is the paired one of k_z_v:
// butterfly f = 2 d + parity of tile (E / O) position 8 d holds kz = f + m Nz/8.
template <typename T, int LNZ, int TY, int NT>
__global__ void __launch_bounds__(NT, 1) k_z_eo_v(GeoV g, int q0, int nq, CQ<T>* W2, const typename kchunks<T>::V* __restrict__ K,
                                                 const int* __restrict__ yslot, TwSet<T> tw, const CQ<T>* __restrict__ two,
                                                 const __grid_constant__ CUtensorMap tmap)
{
    pdl_enter(g);
    constexpr int NZ = 1 << LNZ, LNH = LNZ - 1, NH = 1 << LNH, B = 3 * TY;
    constexpr int LR1 = LNH - 3, R1 = 1 << LR1, S1 = 8, RF = 8;          // make_sched(LNH, 7): R1 . 8
    constexpr int PE = tile_pe(B, 0);
    constexpr int OPAD = TY;         // quads of padding in front of the O tile: in the fused pass a quarter-warp holds one E and one
                                     // O butterfly (TY quads each); without it both fall into the same banks (NH * B * 16 B = 0 mod 128)
    constexpr int NPAIR = S1 * B, PER_ROUND = NT / 2;
    static_assert(NPAIR % 16 == 0 && NT % 32 == 0 && NT % TY == 0 && TY >= 4, "k_z_eo_v: tile shape");
    CQ<T>* s = reinterpret_cast<CQ<T>*>(smem_v2);                        // E tile: points [0, NH), O tile: [NH, 2 NH)
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const bool odd = lane >= 16;
    const int tilesY = g.Ny / TY;
    const int pyt = blockIdx.x % tilesY, ql = blockIdx.x / tilesY;
    const int py0 = pyt * TY;
    const size_t cstride = (size_t)nq * g.nz * g.Ny;
    CQ<T>* base = W2 + (size_t)ql * g.nz * g.Ny + py0;
    const int Ny = g.Ny;
    if (g.pf && blockIdx.x + g.pf < gridDim.x) {                         // next tile's field rows and spectrum rows into L2
        const int bn = blockIdx.x + g.pf, pytn = bn % tilesY, qln = bn / tilesY;
        const CQ<T>* bnx = W2 + (size_t)qln * g.nz * g.Ny + pytn * TY;
        if (g.pft) { if (tid == 0) pf_l2_tensor(&tmap, pytn * TY * 4, 0, qln, 0); }
        else for (int r = tid; r < 3 * g.nz; r += NT) { const int c = r / g.nz, z = r - c * g.nz; pf_l2_span(bnx + c * cstride + (size_t)z * Ny, (uint32_t)(TY * sizeof(CQ<T>))); }
        if (tid >= NT - 2) {
            const int sl = __ldg(yslot + pytn * TY + (tid == NT - 1 ? TY - 1 : 0)) & 0x7fffffff;
            const uint32_t kb = (uint32_t)(g.kpz * kchunks<T>::N * TY * sizeof(typename kchunks<T>::V));
            pf_l2_bulk(K + ((size_t)(q0 + qln) * g.kst + sl / TY) * g.kpz * (kchunks<T>::N * TY), kb);
        }
    }
    float sy;
    const size_t slot = kslot<TY, kchunks<T>::N>(yslot, py0 + tid % TY, g.kpz, sy);
    const CQ<T>* tab = tw.p[0];                                          // w_NH^(i m), [(m - 1) * 8 + i]
    // ---- first pass of both half transforms, inputs straight from global (all nz = NH of them: nothing is padded here)
    for (int qb = wid * 16; qb < NPAIR; qb += PER_ROUND) {
        const int q = qb + (lane & 15), b = q % B, i = q / B;
        const int c = b / TY, ty = b - c * TY;
        const CQ<T>* col = base + c * cstride + ty;
        CQ<T> a[R1];
#pragma unroll
        for (int r = 0; r < R1; ++r) a[r] = ldsq(col + (size_t)(i + S1 * r) * Ny);
        if (odd) {
#pragma unroll
            for (int r = 0; r < R1; ++r) a[r] = cmul(a[r], ldgq(two + i + S1 * r));
        }
        dftR<LR1, false, false>(a);
        CQ<T>* d = s + tile_addr<PE>((odd ? NH : 0) + i, b) + (odd ? OPAD : 0);
        stq(d, a[0]);
#pragma unroll
        for (int m = 1; m < R1; ++m) stq(d + tile_leg<PE, S1>(m), cmul(a[m], ldgq(tab + ((m - 1) << 3) + i)));
    }
    __syncthreads();
    {   // ---- fused pass (k_z_v's paired form): unit u = butterflies (u, W - u), unit 0 = (0, W/2)
        constexpr int W = NZ >> 3, UNITS = (W / 2) * TY, ROW = kchunks<T>::N * TY;
        const typename kchunks<T>::V* Kcol = K + (size_t)(q0 + ql) * g.kst * g.kpz * (kchunks<T>::N * TY) + slot;
        auto pos_of = [](int f) { return (f & 1) * NH + (f >> 1) * 8; };
        auto pad_of = [](int p0) { return p0 >= NH ? OPAD : 0; };
        auto load_fwd = [&](CQ<T> (*a)[RF], int p0, int ty) {
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) {
#pragma unroll
                for (int m = 0; m < RF; ++m) a[cc][m] = ldq(s + tile_addr<PE>(p0, cc * TY + ty) + pad_of(p0) + tile_leg<PE, 1>(m));
                dftR<3, false, false>(a[cc]);
            }
        };
        auto inv_store = [&](CQ<T> (*a)[RF], int p0, int ty) {
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) {
                dftR<3, true, false>(a[cc]);
#pragma unroll
                for (int m = 0; m < RF; ++m) stq(s + tile_addr<PE>(p0, cc * TY + ty) + pad_of(p0) + tile_leg<PE, 1>(m), a[cc][m]);
            }
        };
        auto ksel = [](bool c, const KQ<T>& x, const KQ<T>& y) {
            KQ<T> r;
            r.xx = c ? x.xx : y.xx; r.yy = c ? x.yy : y.yy; r.zz = c ? x.zz : y.zz; r.xy = c ? x.xy : y.xy; r.xz = c ? x.xz : y.xz; r.yz = c ? x.yz : y.yz;
            return r;
        };
#pragma unroll 1
        for (int t = tid; t < UNITS; t += NT) {
            const int ty = t % TY, u = t / TY;
            const bool self = u == 0;
            const int fA = u, fB = self ? W / 2 : W - u;
            KQ<T> KA[4], KB[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) { KA[j] = ldk<TY>(Kcol + (fA + j * W) * ROW); KB[j] = ldk<TY>(Kcol + (fB + j * W) * ROW); }
            const KQ<T> KN = ldk<TY>(Kcol + (self ? 4 * W : fB + 3 * W) * ROW);
            CQ<T> a[3][RF];
            {
                const int p0 = pos_of(fA);
                load_fwd(a, p0, ty);
#pragma unroll
                for (int m = 0; m < 4; ++m) apply_kernel<1>(KA[m], a[0][m], a[1][m], a[2][m], (T)1, (T)sy);
                apply_kernel<0>(ksel(self, KN, KB[3]), a[0][4], a[1][4], a[2][4], self ? (T)1 : (T)-1, (T)sy);
#pragma unroll
                for (int m = 5; m < 8; ++m) apply_kernel<-1>(ksel(self, KA[8 - m], KB[7 - m]), a[0][m], a[1][m], a[2][m], (T)1, (T)sy);
                inv_store(a, p0, ty);
            }
            {
                const int p0 = pos_of(fB);
                load_fwd(a, p0, ty);
#pragma unroll
                for (int m = 0; m < 4; ++m) apply_kernel<1>(KB[m], a[0][m], a[1][m], a[2][m], (T)1, (T)sy);
#pragma unroll
                for (int m = 4; m < 8; ++m) apply_kernel<-1>(ksel(self, KB[7 - m], KA[7 - m]), a[0][m], a[1][m], a[2][m], (T)1, (T)sy);
                inv_store(a, p0, ty);
            }
        }
    }
    __syncthreads();
    // ---- last pass of both half inverses; the E lane finishes z = i + 8 r for r < R1/2, the O lane for r >= R1/2
    for (int qb = wid * 16; qb < NPAIR; qb += PER_ROUND) {
        const int q = qb + (lane & 15), b = q % B, i = q / B;
        const int c = b / TY, ty = b - c * TY;
        CQ<T>* col = base + c * cstride + ty;
        const CQ<T>* d = s + tile_addr<PE>((odd ? NH : 0) + i, b) + (odd ? OPAD : 0);
        CQ<T> a[R1];
        a[0] = ldq(d);
#pragma unroll
        for (int m = 1; m < R1; ++m) a[m] = cmulc(ldq(d + tile_leg<PE, S1>(m)), ldgq(tab + ((m - 1) << 3) + i));
        dftR<LR1, true, false>(a);
        if (odd) {
#pragma unroll
            for (int r = 0; r < R1; ++r) a[r] = cmulc(a[r], ldgq(two + i + S1 * r));
        }
#pragma unroll
        for (int j = 0; j < R1 / 2; ++j) {
            const CQ<T> give = odd ? a[j] : a[j + R1 / 2], keep = odd ? a[j + R1 / 2] : a[j];
            CQ<T> got;
            got.re.x = __shfl_xor_sync(0xffffffffu, give.re.x, 16); got.re.y = __shfl_xor_sync(0xffffffffu, give.re.y, 16);
            got.im.x = __shfl_xor_sync(0xffffffffu, give.im.x, 16); got.im.y = __shfl_xor_sync(0xffffffffu, give.im.y, 16);
            stq(col + (size_t)(i + S1 * (j + (odd ? R1 / 2 : 0))) * Ny, cadd(keep, got));
        }
    }
    pdl_leave(g);
}

// =========================================================================================== K1v / K5v: x stage
// A tile = RP pairs of consecutive y rows of one (component, z); the two rows of a pair are the two lines of a quad.
// The real rows are transformed as packed complex sequences z[m] = x[2m] + i x[2m+1] of length Lc (upper half
// zero: the padding), then split into the real transform's bins k and Lc-k together:
//   2 X[k] = A - i w^k D,  2 X[Lc-k] = conj(A + i w^k D),  A = Z[k] + conj Z[Lc-k],  D = Z[k] - conj Z[Lc-k],
// w = exp(-2 pi i / 2Lc).  The factor 2 is folded into the stored kernel spectrum.

// w^k of the real-transform split, k = 0..Lc/2.  Long rows: w^k = w^(k & ~63) w^(k & 63) from 33 + 64 entries of the
// table (they stay in L1) instead of one read of a 33 KB table per tile.
template <int LLC, typename T> __device__ __forceinline__ CQ<T> split_tw(const CQ<T>* __restrict__ twpost, int k)
{
    if (LLC < 10) return ldgq(twpost + k);
    return cmul(ldgq(twpost + (k & ~63)), ldgq(twpost + (k & 63)));
}

// x R2C FFT fused with the zero padding and the transposition to y-contiguous storage
// (PAPER.md:35, :296-300 xFFT_R2C; :343 "xy transposition ... to avoid strided y FFTs"):  M -> W1v
template <typename T, int LLC, int POL, int RP, int NT, bool SH, bool EMB = false>
__device__ __forceinline__ void x_r2c_body(const GeoV& g, const T* __restrict__ M, CQ<T>* __restrict__ W1,
                                           const ShardMap<T>* map, const TwSet<T>& tw, const CQ<T>* __restrict__ twpost)
{
    using V = typename vec2<T>::type;
    constexpr int LC = 1 << LLC, PITCH = tile_pe(RP | 1, (RP < 8 && skew_ok(LLC, POL)) ? RP : 0, true);
    constexpr Sched SC = make_sched(LLC, POL);
    CQ<T>* s = reinterpret_cast<CQ<T>*>(smem_v2);
    const int tid = threadIdx.x;
    const int tilesY = g.ny / (2 * RP);
    const int ty = blockIdx.x % tilesY, cz = blockIdx.x / tilesY;
    const int y0 = ty * 2 * RP;
    const int c = cz / g.nz, z = cz - c * g.nz;
    // caller's array [3][onz][ony][onx] (= the transform mesh unless embedded); cells outside it are zeros
    const int onx = g.onx, ony = g.ony;
    const bool zin = z < g.onz;
    const T* rows = M + (((size_t)c * g.onz + z) * ony + y0) * onx;
    if (g.pf && tid == 0 && blockIdx.x + g.pf < gridDim.x && onx == g.nx && ony == g.ny)
        pf_l2_bulk(M + (size_t)(blockIdx.x + g.pf) * (2 * RP) * onx, (uint32_t)(2 * RP * onx * sizeof(T)));
    auto ld = [&](int b, int m) {
        V r0, r1;
        if (EMB) {      // embedded mesh: cells outside the caller's array are zeros (only these plans pay for the tests)
            const bool xin = zin && 2 * m < onx;
            r0.x = r0.y = r1.x = r1.y = (T)0;
            if (xin && y0 + 2 * b < ony) r0 = __ldg(reinterpret_cast<const V*>(rows + (size_t)(2 * b) * onx + 2 * m));
            if (xin && y0 + 2 * b + 1 < ony) r1 = __ldg(reinterpret_cast<const V*>(rows + (size_t)(2 * b + 1) * onx + 2 * m));
        } else {
            r0 = __ldg(reinterpret_cast<const V*>(rows + (size_t)(2 * b) * onx + 2 * m));
            r1 = __ldg(reinterpret_cast<const V*>(rows + (size_t)(2 * b + 1) * onx + 2 * m));
        }
        CQ<T> q; q.re.x = r0.x; q.re.y = r1.x; q.im.x = r0.y; q.im.y = r1.y; return q;
    };
    pass_first<T, LLC, POL, RP, PITCH, NT, false>(s, tw.p[0], tid, ld);
    __syncthreads();
    FwdPasses<T, LLC, POL, 1, SC.n, RP, PITCH, NT>::run(s, tw, tid);
    const size_t plane = (size_t)g.nz * g.ny;
    CQ<T>* out = SH ? nullptr : W1 + ((size_t)c * g.hq * g.nz + z) * g.ny + y0;
    constexpr int TOT = (LC / 2 + 1) * RP;
#pragma unroll 2
    for (int t = tid; t < TOT; t += NT) {
        const int b = t % RP, k = t / RP;
        const CQ<T> Zk = ldq(s + tile_addr<PITCH>(pos_of_freq_rt<LLC, POL>(k), b));
        const CQ<T> Zm = ldq(s + tile_addr<PITCH>(pos_of_freq_rt<LLC, POL>((LC - k) & (LC - 1)), b));
        const CQ<T> w = split_tw<LLC>(twpost, k);
        CQ<T> D; D.re = vsub(Zk.re, Zm.re); D.im = vadd(Zk.im, Zm.im);
        const V A = vadd(Zk.re, Zm.re), Bm = vsub(Zk.im, Zm.im);
        const CQ<T> u = cmul(D, w);
        const V xkr = vadd(A, u.im), xki = vsub(Bm, u.re), xmr = vsub(A, u.im), xmi = vneg(vadd(Bm, u.re));
        CQ<T> o0, o1;
        o0.re.x = xkr.x; o0.re.y = xmr.x; o0.im.x = xki.x; o0.im.y = xmi.x;
        o1.re.x = xkr.y; o1.re.y = xmr.y; o1.im.x = xki.y; o1.im.y = xmi.y;
        CQ<T>* d;
        if constexpr (SH) {      // pair k belongs to rank s = k / per: its W1in holds [c][nq_s][nz][ny] (Transfer_S1_to_S2)
            const int sr = min(k / map->per, map->G - 1), k0 = sr * map->per;
            const int nqs = sr == map->G - 1 ? map->total - k0 : map->per;
            d = map->base[sr] + (((size_t)c * nqs + (k - k0)) * g.nz + z) * map->pitch + map->off + y0 + 2 * b;
        } else d = out + (size_t)k * plane + 2 * b;
        stq2(d, o0, o1);
    }
}
template <typename T, int LLC, int POL, int RP, int NT>
__global__ void __launch_bounds__(NT) k_x_r2c_v(GeoV g, const T* __restrict__ M, CQ<T>* __restrict__ W1,
                                               TwSet<T> tw, const CQ<T>* __restrict__ twpost)
{
    pdl_enter(g);
    x_r2c_body<T, LLC, POL, RP, NT, false>(g, M, W1, nullptr, tw, twpost);
    pdl_leave(g);
}
// the same reading an embedded (smaller, any even nx) caller array
template <typename T, int LLC, int POL, int RP, int NT>
__global__ void __launch_bounds__(NT) k_x_r2c_e_v(GeoV g, const T* __restrict__ M, CQ<T>* __restrict__ W1,
                                                 TwSet<T> tw, const CQ<T>* __restrict__ twpost)
{
    pdl_enter(g);
    x_r2c_body<T, LLC, POL, RP, NT, false, true>(g, M, W1, nullptr, tw, twpost);
    pdl_leave(g);
}
// the same on this rank's rows only (g.ny = rows of this rank), every pair stored at the rank that owns it
template <typename T, int LLC, int POL, int RP, int NT>
__global__ void __launch_bounds__(NT) k_x_r2c_sh_v(GeoV g, const T* __restrict__ M, const __grid_constant__ ShardMap<T> map,
                                                  TwSet<T> tw, const CQ<T>* __restrict__ twpost)
{
    pdl_enter(g);
    x_r2c_body<T, LLC, POL, RP, NT, true>(g, M, nullptr, &map, tw, twpost);
    pdl_leave(g);
}

// x C2R FFT fused with the crop; writes H:  W1v -> H
//   2 Z[k] = A + i u,  2 Z[Lc-k] = conj(A - i u),  A = X[k] + conj X[Lc-k],  u = conj(w^k) (X[k] - conj X[Lc-k])
template <typename T, int LLC, int POL, int RP, int NT, bool EMB>
__device__ __forceinline__ void x_c2r_body(const GeoV& g, const CQ<T>* __restrict__ W1, T* __restrict__ H,
                                           const TwSet<T>& tw, const CQ<T>* __restrict__ twpost, const CUtensorMap& tmap)
{
    using V = typename vec2<T>::type;
    constexpr int LC = 1 << LLC, PITCH = tile_pe(RP | 1, (RP < 8 && skew_ok(LLC, POL)) ? RP : 0, true);
    constexpr Sched SC = make_sched(LLC, POL);
    CQ<T>* s = reinterpret_cast<CQ<T>*>(smem_v2);
    const int tid = threadIdx.x;
    const int tilesY = g.ny / (2 * RP);
    const int ty = blockIdx.x % tilesY, cz = blockIdx.x / tilesY;
    const int y0 = ty * 2 * RP;
    const int c = cz / g.nz, z = cz - c * g.nz;
    const size_t plane = (size_t)g.nz * g.ny;
    const CQ<T>* in = W1 + ((size_t)c * g.hq * g.nz + z) * g.ny + y0;
    if (g.pf && blockIdx.x + g.pf < gridDim.x) {
        const int bn = blockIdx.x + g.pf, tyn = bn % tilesY, czn = bn / tilesY, cn = czn / g.nz, zn = czn - cn * g.nz;
        const CQ<T>* inn = W1 + ((size_t)cn * g.hq * g.nz + zn) * g.ny + tyn * 2 * RP;
        if (g.pft) { for (int k0 = tid * 256; k0 <= LC / 2; k0 += NT * 256) pf_l2_tensor(&tmap, tyn * 2 * RP * 4, zn, k0, cn); }   // box {2 RP quads, 1, 256 pairs, 1}
        else for (int k = tid; k <= LC / 2; k += NT) pf_l2_span(inn + (size_t)k * plane, (uint32_t)(2 * RP * sizeof(CQ<T>)));
    }
    constexpr int TOT = (LC / 2 + 1) * RP;
    // Hermitian merge of item t = (pair k, row pair b): Z[k], Z[Lc-k] into the tile
    auto merge = [&](int t, const CQ<T>& Q0, const CQ<T>& Q1) {
        const int b = t % RP, k = t / RP;
        V xkr, xmr, xki, xmi;
        xkr.x = Q0.re.x; xkr.y = Q1.re.x; xmr.x = Q0.re.y; xmr.y = Q1.re.y;
        xki.x = Q0.im.x; xki.y = Q1.im.x; xmi.x = Q0.im.y; xmi.y = Q1.im.y;
        const V Ar = vadd(xkr, xmr), Ai = vsub(xki, xmi);
        CQ<T> D; D.re = vsub(xkr, xmr); D.im = vadd(xki, xmi);
        const CQ<T> u = cmulc(D, split_tw<LLC>(twpost, k));
        CQ<T> Zk, Zm;
        Zk.re = vsub(Ar, u.im); Zk.im = vadd(Ai, u.re);
        Zm.re = vadd(Ar, u.im); Zm.im = vsub(u.re, Ai);
        stq(s + tile_addr<PITCH>(pos_of_freq_rt<LLC, POL>(k), b), Zk);
        if (k != 0 && 2 * k != LC) stq(s + tile_addr<PITCH>(pos_of_freq_rt<LLC, POL>(LC - k), b), Zm);
    };
    auto fetch = [&](int t, CQ<T>& Q0, CQ<T>& Q1) {
        const int b = t % RP, k = t / RP;
        const CQ<T>* d = in + (size_t)k * plane + 2 * b;
        if (RP >= 8) { Q0 = ldsq(d); Q1 = ldsq(d + 1); }      // 256-byte runs: two 128-bit loads measured faster (C3)
        else ldq2<(RP >= 4)>(d, Q0, Q1);
    };
    // UB items per thread are requested before the first is used: a warp pays the memory latency TOT / (UB NT) times per
    // tile instead of TOT / (2 NT) times (the merge loop was 36 % of this kernel's stall samples at C3)
    constexpr int UB = 4, FULL = TOT / (UB * NT) * (UB * NT);
#pragma unroll 1
    for (int t0 = tid; t0 < FULL; t0 += UB * NT) {
        CQ<T> Q0[UB], Q1[UB];
#pragma unroll
        for (int u = 0; u < UB; ++u) fetch(t0 + u * NT, Q0[u], Q1[u]);
#pragma unroll
        for (int u = 0; u < UB; ++u) merge(t0 + u * NT, Q0[u], Q1[u]);
    }
#pragma unroll 1
    for (int t = FULL + tid; t < TOT; t += NT) { CQ<T> Q0, Q1; fetch(t, Q0, Q1); merge(t, Q0, Q1); }
    __syncthreads();
    InvPasses<T, LLC, POL, 1, SC.n, RP, PITCH, NT>::run(s, tw, tid);
    const int onx = g.onx, ony = g.ony, acc = g.acc;
    const bool zin = z < g.onz;
    T* rows = H + (((size_t)c * g.onz + z) * ony + y0) * onx;      // caller's array; cells outside it are dropped
    auto st = [&](int b, int m, CQ<T> v) {
        if (EMB && (!zin || 2 * m >= onx)) return;
        V r0, r1; r0.x = v.re.x; r0.y = v.im.x; r1.x = v.re.y; r1.y = v.im.y;
        V* d0 = reinterpret_cast<V*>(rows + (size_t)(2 * b) * onx + 2 * m);
        V* d1 = reinterpret_cast<V*>(rows + (size_t)(2 * b + 1) * onx + 2 * m);
        if (EMB) {
            if (y0 + 2 * b < ony) { if (acc) { const V o0 = *d0; r0.x += o0.x; r0.y += o0.y; } *d0 = r0; }
            if (y0 + 2 * b + 1 < ony) { if (acc) { const V o1 = *d1; r1.x += o1.x; r1.y += o1.y; } *d1 = r1; }
        } else {
            if (acc) { const V o0 = *d0, o1 = *d1; r0.x += o0.x; r0.y += o0.y; r1.x += o1.x; r1.y += o1.y; }
            *d0 = r0; *d1 = r1;
        }
    };
    pass_last<T, LLC, POL, RP, PITCH, NT, false>(s, tw.p[0], tid, st);
}
template <typename T, int LLC, int POL, int RP, int NT>
__global__ void __launch_bounds__(NT) k_x_c2r_v(GeoV g, const CQ<T>* __restrict__ W1, T* __restrict__ H,
                                               TwSet<T> tw, const CQ<T>* __restrict__ twpost, const __grid_constant__ CUtensorMap tmap)
{
    pdl_enter(g);
    x_c2r_body<T, LLC, POL, RP, NT, false>(g, W1, H, tw, twpost, tmap);
    pdl_leave(g);
}
// the same writing an embedded caller array (the crop of the cells outside it)
template <typename T, int LLC, int POL, int RP, int NT>
__global__ void __launch_bounds__(NT) k_x_c2r_e_v(GeoV g, const CQ<T>* __restrict__ W1, T* __restrict__ H,
                                                 TwSet<T> tw, const CQ<T>* __restrict__ twpost, const __grid_constant__ CUtensorMap tmap)
{
    pdl_enter(g);
    x_c2r_body<T, LLC, POL, RP, NT, true>(g, W1, H, tw, twpost, tmap);
    pdl_leave(g);
}

}  // namespace v2
}  // namespace demag
