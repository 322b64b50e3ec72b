// vg_kernels.cuh -- the one streaming kernel every (solid, query) pair instantiates.
//
// Layout: six FP64 SoA arrays in, one array out, each track touched once.
// One thread evaluates TPT = 2 consecutive tracks: every input array is read with one 128-bit
// ld.global.nc.L1::no_allocate per thread (a warp reads 512 contiguous bytes per array), the result leaves as
// one 128-bit (64-bit for Inside) streaming store.  The solid's constants arrive by value in kernel-parameter
// space (`__grid_constant__`), so they are warp-uniform constant-bank operands.  A 64-bit-per-track
// instantiation (TPT = 1) serves arrays that are only 8-byte aligned and the odd tail.
#pragma once
#include "vg_shapes.cuh"
#include "vg_tma.cuh"

#include <atomic>

namespace vg {

struct Tracks {
    const double *x, *y, *z, *dx, *dy, *dz;
};

#ifndef VG_BLOCK
#define VG_BLOCK 256
#endif
#ifndef VG_MINB
#define VG_MINB 1
#endif
constexpr int kBlock = VG_BLOCK;
constexpr int64_t kSmallBatchTpt1 = 2 * 148 * 256; // tracks below which two tracks per thread leave SMs without a CTA

extern std::atomic<int64_t> g_launches; // kernel launches made by the library (vg_launch_count)
extern std::atomic<int64_t> g_pdl;      // vg_set_option(VG_OPT_PDL)

// every kernel of the library is launched through this: optional programmatic-dependent-launch attribute
template <class... KArgs, class... Args>
cudaError_t launch_kernel(void (*kern)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t stream,
                          Args &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = g_pdl.load(std::memory_order_relaxed) ? 1 : 0;
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

template <class S, int Q>
VG_DEV void eval_store(const typename S::P &p, double x, double y, double z, double dx, double dy, double dz,
                       double step_max, double &od, int &oi)
{
    if (Q == qInside) {
        oi = S::inside(p, x, y, z);
    } else if (Q == qSafeIn) {
        od = S::safety(p, x, y, z);
    } else if (Q == qSafeOut) {
        od = -S::safety(p, x, y, z);
    } else {
        double t = (Q == qDistIn) ? S::dist_in(p, x, y, z, dx, dy, dz) : S::dist_out(p, x, y, z, dx, dy, dz);
        od = t <= step_max ? t : inf(); // reading R5; -1 passes because step_max >= 0
    }
}

// Per-(solid, query) launch tuning, from the sweeps recorded in DESIGN.md, Appendix A.1:
//   minb   -- minimum resident CTAs per SM of the direct kernel, i.e. its register cap (65536 / (256 minb)).  The
//             straight-line distance code takes ~100 registers if allowed to, which leaves 2 CTAs per SM and too
//             few warps to cover the FP64 latencies; capped at 64 registers (4 CTAs) it runs 15-25 % faster.
//   stream -- VG_FORM_AUTO runs the persistent streaming form (below) instead of the direct one.
//   block  -- CTA size of the direct kernel.  128 threads serve the Tube safeties better at n = 2^20 (1024 tracks per
//             SM-resident CTA pair instead of 512 per CTA: finer hand-out over the 148 SMs, shorter tail).
template <class S, int Q> struct Tune {
    static constexpr int minb = (Q == qDistIn || Q == qDistOut) ? 4 : VG_MINB;
    static constexpr bool stream = false;
    static constexpr int block = kBlock;
};
template <int F> struct Tune<TubeT<F>, qDistIn> {
    static constexpr int minb = 4;
    static constexpr bool stream = true;
    static constexpr int block = kBlock;
};
#ifndef VG_TUBE_SAFE_BLOCK
#define VG_TUBE_SAFE_BLOCK 128
#endif
template <int F> struct Tune<TubeT<F>, qSafeIn> {
    static constexpr int minb = VG_MINB;
    static constexpr bool stream = false;
    static constexpr int block = VG_TUBE_SAFE_BLOCK;
};
template <int F> struct Tune<TubeT<F>, qSafeOut> {
    static constexpr int minb = VG_MINB;
    static constexpr bool stream = false;
    static constexpr int block = VG_TUBE_SAFE_BLOCK;
};
#ifndef VG_CONE_SAFE_BLOCK
#define VG_CONE_SAFE_BLOCK 128
#endif
#ifndef VG_CONE_SAFE_MINB
#define VG_CONE_SAFE_MINB VG_MINB
#endif
template <int F> struct Tune<ConeT<F>, qSafeIn> {
    static constexpr int minb = VG_CONE_SAFE_MINB;
    static constexpr bool stream = false;
    static constexpr int block = VG_CONE_SAFE_BLOCK;
};
template <int F> struct Tune<ConeT<F>, qSafeOut> {
    static constexpr int minb = VG_CONE_SAFE_MINB;
    static constexpr bool stream = false;
    static constexpr int block = VG_CONE_SAFE_BLOCK;
};
// The exact Trd safeties are bound by their FP64 instruction count (about 84 of 134 instructions per track), not by
// the launch shape: the streaming form (128 registers, one resident wave) took 30.9 / 31.5 us at 4 Mi tracks, 256-thread
// direct CTAs 33.0 / 33.9 us, 128-thread direct CTAs capped at 64 registers (8 CTAs per SM, no spills) 28.9 / 30.6 us.
#ifndef VG_TRD_SAFE_BLOCK
#define VG_TRD_SAFE_BLOCK 128
#endif
#ifndef VG_TRD_SAFE_MINB
#define VG_TRD_SAFE_MINB 8
#endif
#ifndef VG_TRD_SAFE_STREAM
#define VG_TRD_SAFE_STREAM false
#endif
template <> struct Tune<Trd, qSafeIn> {
    static constexpr int minb = VG_TRD_SAFE_MINB;
    static constexpr bool stream = VG_TRD_SAFE_STREAM;
    static constexpr int block = VG_TRD_SAFE_BLOCK;
};
template <> struct Tune<Trd, qSafeOut> {
    static constexpr int minb = VG_TRD_SAFE_MINB;
    static constexpr bool stream = VG_TRD_SAFE_STREAM;
    static constexpr int block = VG_TRD_SAFE_BLOCK;
};

template <class S, int Q, int TPT>
__global__ void __launch_bounds__(Tune<S, Q>::block, Tune<S, Q>::minb)
    query_kernel(const __grid_constant__ typename S::P p, Tracks t, double step_max, int64_t n, void *out)
{
    constexpr bool kDir = (Q == qDistIn || Q == qDistOut);
    int64_t i = (int64_t(blockIdx.x) * Tune<S, Q>::block + threadIdx.x) * TPT;
    pdl_launch_dependents();
    pdl_wait();
    if (i >= n) return;
    if (TPT == 2 && i + 1 < n) {
        double2 x = ldg2(t.x + i), y = ldg2(t.y + i), z = ldg2(t.z + i);
        double2 dx = make_double2(0, 0), dy = dx, dz = dx;
        if (kDir) {
            dx = ldg2(t.dx + i);
            dy = ldg2(t.dy + i);
            dz = ldg2(t.dz + i);
        }
        double d0 = 0, d1 = 0;
        int i0 = 0, i1 = 0;
        eval_store<S, Q>(p, x.x, y.x, z.x, dx.x, dy.x, dz.x, step_max, d0, i0);
        eval_store<S, Q>(p, x.y, y.y, z.y, dx.y, dy.y, dz.y, step_max, d1, i1);
        if (Q == qInside)
            stg2i(static_cast<int32_t *>(out) + i, i0, i1);
        else
            stg2(static_cast<double *>(out) + i, d0, d1);
    } else {
        double x = ldg1(t.x + i), y = ldg1(t.y + i), z = ldg1(t.z + i);
        double dx = 0, dy = 0, dz = 0;
        if (kDir) {
            dx = ldg1(t.dx + i);
            dy = ldg1(t.dy + i);
            dz = ldg1(t.dz + i);
        }
        double d0 = 0;
        int i0 = 0;
        eval_store<S, Q>(p, x, y, z, dx, dy, dz, step_max, d0, i0);
        if (Q == qInside)
            stg1i(static_cast<int32_t *>(out) + i, i0);
        else
            stg1(static_cast<double *>(out) + i, d0);
    }
}

// ---- the fused "basket" kernel: all five answers of a track from one pass over its six coordinates ----
//
// A basket of particles in one volume asks all three questions of the paper every step (SURVEY.md
// sec. 8(f) f1).  Five separate launches read 3 x 24 + 2 x 48 = 168 B and write 36 B per track and pay five launch
// latencies; this kernel reads 48 B and writes 36 B once.  The per-solid functions are inlined into one
// straight-line body, so the compiler shares their common subexpressions (rho^2, the classification, the phi terms).
struct AllOut {
    int32_t *cls;
    double *din, *dout, *sin, *sout;
};

#ifndef VG_ALL_MINB
#define VG_ALL_MINB 4
#endif

template <class S>
VG_DEV void eval_all(const typename S::P &p, double x, double y, double z, double dx, double dy, double dz,
                     double step_max, int &cls, double &din, double &dout, double &sdf)
{
    cls = S::inside(p, x, y, z);
    sdf = S::safety(p, x, y, z);
    const double a = S::dist_in(p, x, y, z, dx, dy, dz), b = S::dist_out(p, x, y, z, dx, dy, dz);
    din = a <= step_max ? a : inf();
    dout = b <= step_max ? b : inf();
}

// One track per thread, capped at 64 registers (4 CTAs of 256 threads per SM): the five answers are ~400 instructions of
// dependent FP64 work per track, and what bounds the kernel is the number of warps there are to overlap those chains,
// not its loads.  Two tracks per thread with 128-bit loads (80 registers, 3 CTAs) measured 4-6 % slower for the tube and
// the cone (20.7 -> 19.4 us at 1 Mi, 74.2 -> 71.2 us at 4 Mi tracks) and the same for the trd.
template <class S>
__global__ void __launch_bounds__(kBlock, VG_ALL_MINB)
    query_all_kernel(const __grid_constant__ typename S::P p, Tracks t, double step_max, int64_t n, AllOut o)
{
    const int64_t i = int64_t(blockIdx.x) * kBlock + threadIdx.x;
    pdl_launch_dependents();
    pdl_wait();
    if (i >= n) return;
    double x = ldg1(t.x + i), y = ldg1(t.y + i), z = ldg1(t.z + i);
    double dx = ldg1(t.dx + i), dy = ldg1(t.dy + i), dz = ldg1(t.dz + i);
    int c0;
    double a0, b0, s0;
    eval_all<S>(p, x, y, z, dx, dy, dz, step_max, c0, a0, b0, s0);
    stg1i(o.cls + i, c0);
    stg1(o.din + i, a0);
    stg1(o.dout + i, b0);
    stg1(o.sin + i, s0);
    stg1(o.sout + i, -s0);
}

template <class S>
cudaError_t launch_all(const typename S::P &p, const Tracks &t, double step_max, int64_t n, const AllOut &o, bool vec,
                       cudaStream_t stream)
{
    (void)vec; // any alignment
    if (n <= 0) return cudaSuccess;
    unsigned grid = unsigned((n + kBlock - 1) / kBlock);
    return launch_kernel(query_all_kernel<S>, grid, kBlock, 0, stream, p, t, step_max, n, o);
}

// ---- the pipelined form of the same kernel (the default for 16-byte aligned arrays and n >= g_pipe_min_n) ----
//
// Why: the plain kernel above keeps a thread's loads in flight only until its own arithmetic starts; with 60-90
// registers per thread (tube / cone / trd / polycone distances) the SM holds 2-3 CTAs, whose load and compute
// phases do not overlap well: ncu showed DRAM and the FP64 pipe BOTH at 35-55 % (profiles/r1_*).  Here the track
// tiles travel global -> shared memory as TMA bulk copies (cp.async.bulk, one 4 KiB copy per SoA array per tile)
// issued by a producer warp into a kStages-deep ring guarded by full/empty mbarriers; kPipeWarps consumer warps
// take two tracks per thread out of the ring with 128-bit shared loads, hand the slot back at once and evaluate.
// The grid has one CTA per tile, but the CTAs that get to run are persistent: the producer takes over the block
// index of a not yet launched CTA with cluster launch control (clusterlaunchcontrol.try_cancel, sm_100) for every
// further tile, so tiles are handed out dynamically by the hardware scheduler (a static round-robin left the SMs
// finishing 50 % apart, profiles/r1_*) and the ring never drains between tiles.  The bytes in flight per SM are set
// by the ring (up to kStages x 24 KiB per CTA), not by the register file, and loads of later tiles overlap the
// FP64 work of the current one.  Results leave as 128-bit streaming stores straight from registers.
#ifndef VG_PIPE_WARPS
#define VG_PIPE_WARPS 8
#endif
#ifndef VG_PIPE_STAGES
#define VG_PIPE_STAGES 4
#endif
#ifndef VG_PIPE_MINB
#define VG_PIPE_MINB 2
#endif
constexpr int kPipeWarps = VG_PIPE_WARPS;
constexpr int kPipeStages = VG_PIPE_STAGES;
constexpr int kPipeThreads = 32 * kPipeWarps + 32; // + the producer warp
constexpr int kPipeTile = 64 * kPipeWarps;         // tracks per tile: two per consumer thread

extern std::atomic<int64_t> g_pipe_min_n; // vg_set_option(VG_OPT_PIPE_MIN_N)
extern std::atomic<int64_t> g_host_chunk; // vg_set_option(VG_OPT_HOST_CHUNK): tracks per chunk of the host-fed pipeline, 0 = auto
extern std::atomic<int64_t> g_nav_form;   // vg_set_option(VG_OPT_NAV_FORM): 0 auto, 1 per-lane, 2 warp-cooperative phase 2 of ComputeStep
extern std::atomic<int64_t> g_form;       // vg_set_option(VG_OPT_FORM): 0 auto, 1 direct, 2 pipelined, 3 streaming

// VG_FORM_AUTO: the pairs whose pipelined form measured faster than the direct one at n >= 2^22 (profiles/):
// only the heaviest straight-line kernel, where the direct form's registers leave too few warps to overlap its
// loads with its FP64 work.  Everything lighter is faster direct (no ring hand-offs, four to eight CTAs per SM).
template <class S, int Q> struct PipeByDefault { static constexpr bool value = false; };

template <class S, int Q>
__global__ void __launch_bounds__(kPipeThreads, VG_PIPE_MINB)
    query_pipe_kernel(const __grid_constant__ typename S::P p, Tracks t, double step_max, int64_t n, void *out)
{
    constexpr bool kDir = (Q == qDistIn || Q == qDistOut);
    constexpr int kArr = kDir ? 6 : 3;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *ring = reinterpret_cast<double *>(smem_raw); // [kPipeStages][kArr][kPipeTile]
    __shared__ __align__(16) unsigned char clc_resp[16];
    __shared__ __align__(8) uint64_t full[kPipeStages], empty[kPipeStages], clc_bar;
    __shared__ int tile_of[kPipeStages];
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < kPipeStages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], kPipeWarps);
        }
        mbar_init(&clc_bar, 1);
        mbar_fence_init();
    }
    pdl_launch_dependents();
    __syncthreads();
    pdl_wait(); // nothing above touches global memory: it overlaps the tail of the previous kernel in the stream
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (warp == kPipeWarps) { // producer: one elected lane schedules tiles and feeds the ring
        if (lane != 0) return;
        const double *src[6] = { t.x, t.y, t.z, t.dx, t.dy, t.dz };
        int s = 0, tile = blockIdx.x;
        uint32_t ph = 1; // a fresh `empty` barrier lets the wait on parity 1 pass: every slot starts free
        uint32_t clc_ph = 0;
        while (true) {
            // ask the hardware for the next tile (a not yet launched CTA of this grid) while this one is issued
            mbar_expect_tx(&clc_bar, 16);
            clc_try_cancel(clc_resp, &clc_bar);
            mbar_wait(&empty[s], ph);
            tile_of[s] = tile;
            const int64_t base = int64_t(tile) * kPipeTile;
            const int64_t left = n - base;
            const uint32_t cnt = left < kPipeTile ? uint32_t(left) : uint32_t(kPipeTile);
            const uint32_t bytes = (cnt * 8u) & ~15u; // an odd last track is read by its consumer straight from global
            if (bytes) {
                mbar_expect_tx(&full[s], kArr * bytes);
#pragma unroll
                for (int a = 0; a < kArr; ++a) bulk_g2s(ring + (s * kArr + a) * kPipeTile, src[a] + base, bytes, &full[s]);
            } else {
                mbar_arrive(&full[s]);
            }
            if (++s == kPipeStages) {
                s = 0;
                ph ^= 1u;
            }
            mbar_wait(&clc_bar, clc_ph);
            clc_ph ^= 1u;
            tile = clc_decode_x(clc_resp);
            fence_proxy_async_smem(); // the next response may overwrite clc_resp
            if (tile < 0) break;
        }
        mbar_wait(&empty[s], ph); // end marker for the consumers
        tile_of[s] = -1;
        mbar_arrive(&full[s]);
        return;
    }

    int s = 0;
    uint32_t ph = 0;
    while (true) {
        mbar_wait(&full[s], ph);
        const int tile = tile_of[s];
        if (tile < 0) break;
        const int64_t i = int64_t(tile) * kPipeTile + 2 * threadIdx.x;
        const bool pair = i + 1 < n;
        const double *st = ring + s * kArr * kPipeTile + 2 * threadIdx.x;
        double2 x = make_double2(0, 0), y = x, z = x, dx = x, dy = x, dz = x;
        if (pair) {
            x = *reinterpret_cast<const double2 *>(st);
            y = *reinterpret_cast<const double2 *>(st + kPipeTile);
            z = *reinterpret_cast<const double2 *>(st + 2 * kPipeTile);
            if (kDir) {
                dx = *reinterpret_cast<const double2 *>(st + 3 * kPipeTile);
                dy = *reinterpret_cast<const double2 *>(st + 4 * kPipeTile);
                dz = *reinterpret_cast<const double2 *>(st + 5 * kPipeTile);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]); // the slot is free again as soon as the warp holds its tracks in registers
        if (++s == kPipeStages) {
            s = 0;
            ph ^= 1u;
        }
        if (pair) {
            double d0 = 0, d1 = 0;
            int i0 = 0, i1 = 0;
            eval_store<S, Q>(p, x.x, y.x, z.x, dx.x, dy.x, dz.x, step_max, d0, i0);
            eval_store<S, Q>(p, x.y, y.y, z.y, dx.y, dy.y, dz.y, step_max, d1, i1);
            if (Q == qInside)
                stg2i(static_cast<int32_t *>(out) + i, i0, i1);
            else
                stg2(static_cast<double *>(out) + i, d0, d1);
        } else if (i < n) { // odd last track
            double x1 = ldg1(t.x + i), y1 = ldg1(t.y + i), z1 = ldg1(t.z + i);
            double dx1 = 0, dy1 = 0, dz1 = 0;
            if (kDir) {
                dx1 = ldg1(t.dx + i);
                dy1 = ldg1(t.dy + i);
                dz1 = ldg1(t.dz + i);
            }
            double d0 = 0;
            int i0 = 0;
            eval_store<S, Q>(p, x1, y1, z1, dx1, dy1, dz1, step_max, d0, i0);
            if (Q == qInside)
                stg1i(static_cast<int32_t *>(out) + i, i0);
            else
                stg1(static_cast<double *>(out) + i, d0);
        }
    }
}

// ---- the persistent streaming form: one resident wave of CTAs, each owning ONE contiguous range of track pairs ----
//
// Why: with one CTA per 512 tracks the direct form runs n / 512 CTAs in waves of (SM count x CTAs per SM); at
// n = 2^20 that is 2048 CTAs over e.g. 444 resident ones = 4.6 waves, so the last wave leaves 40 % of the SMs idle,
// and inside a wave the CTAs of an SM load and compute in step.  Here the grid is exactly one resident wave, every
// CTA gets the same number of pairs (rounded to a warp's 512-byte row), so every SM has the same work to within
// one row, and each thread issues the 128-bit loads of its NEXT pair before it evaluates the current one (register
// double buffering): the loads of iteration i+1 are in flight during the FP64 work of iteration i.
#ifndef VG_SBLOCK
#define VG_SBLOCK 256
#endif
#ifndef VG_SMINB
#define VG_SMINB 2
#endif
constexpr int kSBlock = VG_SBLOCK;

template <class S, int Q>
__global__ void __launch_bounds__(kSBlock, VG_SMINB)
    query_stream_kernel(const __grid_constant__ typename S::P p, Tracks t, double step_max, int64_t n, void *out,
                        int64_t pairs_per_cta)
{
    constexpr bool kDir = (Q == qDistIn || Q == qDistOut);
    using S_ = S;
    pdl_launch_dependents();
    pdl_wait();
    const int64_t npairs = n >> 1;
    const int64_t lo = int64_t(blockIdx.x) * pairs_per_cta;
    const int64_t hi = lo + pairs_per_cta < npairs ? lo + pairs_per_cta : npairs;
    int64_t j = lo + threadIdx.x;
    // two register sets used in turn (the loop is unrolled by two so that no set is ever copied)
    double2 xa = make_double2(0, 0), ya = xa, za = xa, dxa = xa, dya = xa, dza = xa;
    double2 xb = xa, yb = xa, zb = xa, dxb = xa, dyb = xa, dzb = xa;
#define VG_LOAD_PAIR(S, J)                                                                                           \
    do {                                                                                                             \
        x##S = ldg2(t.x + 2 * (J)), y##S = ldg2(t.y + 2 * (J)), z##S = ldg2(t.z + 2 * (J));                          \
        if (kDir) dx##S = ldg2(t.dx + 2 * (J)), dy##S = ldg2(t.dy + 2 * (J)), dz##S = ldg2(t.dz + 2 * (J));          \
    } while (0)
#define VG_EVAL_PAIR(S, J)                                                                                           \
    do {                                                                                                             \
        double d0 = 0, d1 = 0;                                                                                       \
        int i0 = 0, i1 = 0;                                                                                          \
        eval_store<S_, Q>(p, x##S.x, y##S.x, z##S.x, dx##S.x, dy##S.x, dz##S.x, step_max, d0, i0);                   \
        eval_store<S_, Q>(p, x##S.y, y##S.y, z##S.y, dx##S.y, dy##S.y, dz##S.y, step_max, d1, i1);                   \
        if (Q == qInside)                                                                                            \
            stg2i(static_cast<int32_t *>(out) + 2 * (J), i0, i1);                                                    \
        else                                                                                                         \
            stg2(static_cast<double *>(out) + 2 * (J), d0, d1);                                                      \
    } while (0)
    if (j < hi) VG_LOAD_PAIR(a, j);
    while (j < hi) {
        if (j + kSBlock < hi) VG_LOAD_PAIR(b, j + kSBlock);
        VG_EVAL_PAIR(a, j);
        j += kSBlock;
        if (j >= hi) break;
        if (j + kSBlock < hi) VG_LOAD_PAIR(a, j + kSBlock);
        VG_EVAL_PAIR(b, j);
        j += kSBlock;
    }
#undef VG_LOAD_PAIR
#undef VG_EVAL_PAIR
    if ((n & 1) && blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) { // odd last track
        const int64_t i = n - 1;
        double x1 = ldg1(t.x + i), y1 = ldg1(t.y + i), z1 = ldg1(t.z + i);
        double dx1 = 0, dy1 = 0, dz1 = 0;
        if (kDir) dx1 = ldg1(t.dx + i), dy1 = ldg1(t.dy + i), dz1 = ldg1(t.dz + i);
        double d0 = 0;
        int i0 = 0;
        eval_store<S, Q>(p, x1, y1, z1, dx1, dy1, dz1, step_max, d0, i0);
        if (Q == qInside)
            stg1i(static_cast<int32_t *>(out) + i, i0);
        else
            stg1(static_cast<double *>(out) + i, d0);
    }
}

// resident CTAs of the streaming kernel on the current device (queried once per device and instantiation)
template <class S, int Q> cudaError_t stream_capacity(int *cap)
{
    constexpr int kMaxDev = 64;
    static std::atomic<int> cached[kMaxDev];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < kMaxDev && (*cap = cached[dev].load(std::memory_order_acquire)) > 0) return cudaSuccess;
    int sms = 0, per_sm = 0;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, query_stream_kernel<S, Q>, kSBlock, 0)) != cudaSuccess)
        return e;
    *cap = sms * (per_sm < 1 ? 1 : per_sm);
    if (dev >= 0 && dev < kMaxDev) cached[dev].store(*cap, std::memory_order_release);
    return cudaSuccess;
}

// resident CTAs of the pipelined kernel on the current device (configured once per device and instantiation)
template <class S, int Q> cudaError_t pipe_capacity(int *cap, size_t *smem_out)
{
    constexpr int kMaxDev = 64;
    constexpr int kArr = (Q == qDistIn || Q == qDistOut) ? 6 : 3;
    constexpr size_t smem = size_t(kPipeStages) * kArr * kPipeTile * sizeof(double);
    static std::atomic<int> cached[kMaxDev];
    *smem_out = smem;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < kMaxDev && (*cap = cached[dev].load(std::memory_order_acquire)) > 0) return cudaSuccess;
    int sms = 0, per_sm = 0;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(query_pipe_kernel<S, Q>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem))) != cudaSuccess)
        return e;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, query_pipe_kernel<S, Q>, kPipeThreads, smem)) != cudaSuccess)
        return e;
    *cap = sms * (per_sm < 1 ? 1 : per_sm);
    if (dev >= 0 && dev < kMaxDev) cached[dev].store(*cap, std::memory_order_release);
    return cudaSuccess;
}

// G = the run-time-flag form of the solid (pipelined kernel), S = the specialisation picked from the flags
template <class G, class S, int Q>
cudaError_t launch_query(const typename S::P &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                         cudaStream_t stream)
{
    if (n <= 0) return cudaSuccess;
#ifdef VG_FORCE_TPT1
    vec = false;
#endif
    const int64_t form = g_form.load(std::memory_order_relaxed);
    // a batch too small to give every SM a CTA at two tracks per thread runs one track per thread: twice the CTAs
    // (configs[0], 65,536 tracks: 128 -> 256 CTAs of 256 threads on 148 SMs; DistanceToOut 2.35 -> 2.26 us, safeties 1.88 -> 1.80 us)
    if (form == 0 && n < kSmallBatchTpt1) vec = false;
    const bool pipe = form == 2 || (form == 0 && PipeByDefault<G, Q>::value);
    if (vec && pipe && n >= g_pipe_min_n.load(std::memory_order_relaxed)) {
        int cap = 0;
        size_t smem = 0;
        cudaError_t e = pipe_capacity<G, Q>(&cap, &smem);
        if (e != cudaSuccess) return e;
        (void)cap;
        int64_t tiles = (n + kPipeTile - 1) / kPipeTile; // one CTA per tile; running CTAs cancel and take over pending ones
        return launch_kernel(query_pipe_kernel<G, Q>, unsigned(tiles), kPipeThreads, smem, stream, p, t, step_max, n, out);
    }
    if (vec && n >= 2 && (form == 3 || (form == 0 && Tune<S, Q>::stream))) {
        int cap = 0;
        cudaError_t e = stream_capacity<S, Q>(&cap);
        if (e != cudaSuccess) return e;
        const int64_t npairs = n >> 1;
        int64_t grid = (npairs + kSBlock - 1) / kSBlock;
        if (grid > cap) grid = cap;
        int64_t per = (npairs + grid - 1) / grid;
        per = (per + 31) / 32 * 32; // a warp's row of 32 pairs = 512 contiguous bytes per array
        grid = (npairs + per - 1) / per;
        return launch_kernel(query_stream_kernel<S, Q>, unsigned(grid), kSBlock, 0, stream, p, t, step_max, n, out, per);
    }
    constexpr int kB = Tune<S, Q>::block;
    if (vec) {
        int64_t threads = (n + 1) / 2;
        unsigned grid = unsigned((threads + kB - 1) / kB);
        return launch_kernel(query_kernel<S, Q, 2>, grid, kB, 0, stream, p, t, step_max, n, out);
    }
    unsigned grid = unsigned((n + kB - 1) / kB);
    return launch_kernel(query_kernel<S, Q, 1>, grid, kB, 0, stream, p, t, step_max, n, out);
}

template <class G, class S = G>
cudaError_t launch_any(int q, const typename S::P &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                       cudaStream_t stream)
{
    switch (q) {
    case qInside: return launch_query<G, S, qInside>(p, t, step_max, n, out, vec, stream);
    case qDistIn: return launch_query<G, S, qDistIn>(p, t, step_max, n, out, vec, stream);
    case qDistOut: return launch_query<G, S, qDistOut>(p, t, step_max, n, out, vec, stream);
    case qSafeIn: return launch_query<G, S, qSafeIn>(p, t, step_max, n, out, vec, stream);
    case qSafeOut: return launch_query<G, S, qSafeOut>(p, t, step_max, n, out, vec, stream);
    }
    return cudaErrorInvalidValue;
}

// one translation unit per solid defines these (vg_k_<solid>.cu), so the solids compile in parallel
cudaError_t launch_box(int q, const BoxP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                       cudaStream_t s);
cudaError_t launch_orb(int q, const OrbP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                       cudaStream_t s);
cudaError_t launch_tube(int q, const TubeP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                        cudaStream_t s);
cudaError_t launch_cone(int q, const ConeP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                        cudaStream_t s);
cudaError_t launch_trd(int q, const TrdP &p, const Tracks &t, double step_max, int64_t n, void *out, bool vec,
                       cudaStream_t s);
cudaError_t launch_polycone(int q, const PolyconeP &p, const PconGrid &g, const Tracks &t, double step_max, int64_t n,
                            void *out, bool vec, cudaStream_t s);

// the fused five-query kernel of each solid (the polycone has none: its queries run as five launches)
cudaError_t launch_box_all(const BoxP &p, const Tracks &t, double step_max, int64_t n, const AllOut &o, bool vec, cudaStream_t s);
cudaError_t launch_orb_all(const OrbP &p, const Tracks &t, double step_max, int64_t n, const AllOut &o, bool vec, cudaStream_t s);
cudaError_t launch_tube_all(const TubeP &p, const Tracks &t, double step_max, int64_t n, const AllOut &o, bool vec, cudaStream_t s);
cudaError_t launch_cone_all(const ConeP &p, const Tracks &t, double step_max, int64_t n, const AllOut &o, bool vec, cudaStream_t s);
cudaError_t launch_trd_all(const TrdP &p, const Tracks &t, double step_max, int64_t n, const AllOut &o, bool vec, cudaStream_t s);

cudaError_t launch_polycone_all(const PolyconeP &p, const PconGrid &g, const Tracks &t, double step_max, int64_t n, const AllOut &o,
                                bool vec, cudaStream_t s); // cudaErrorNotSupported: run the five queries separately

// navigation (vg_nav.cu)
cudaError_t launch_compute_step(const SolidU &mother, const unsigned char *table_dev, const NavMeta &meta, const Tracks &t,
                                double step_max, int64_t n, double *step, int32_t *hit, cudaStream_t s);
cudaError_t launch_volume_safety(const SolidU &mother, const unsigned char *table_dev, const NavMeta &meta, const Tracks &t, int64_t n,
                                 double *safety, cudaStream_t s);

// boolean solids (vg_bool.cu)
cudaError_t launch_boolean(int q, const BoolP &p, const Tracks &t, double step_max, int64_t n, void *out, cudaStream_t s,
                           bool vec = false);

// booleans with a polycone operand (vg_boolx.cu)
cudaError_t launch_boolx(int q, const BoolP &p, const Tracks &t, double step_max, int64_t n, void *out, cudaStream_t s);

// nested booleans (vg_csg.cu)
cudaError_t launch_csg(int q, const CsgP &p, const Tracks &t, double step_max, int64_t n, void *out, cudaStream_t s);

// hierarchy of volumes (vg_world.cu)
cudaError_t launch_world_locate(const WorldTab &w, const Tracks &t, int64_t n, int32_t *out, cudaStream_t s);
cudaError_t launch_world_step(const WorldTab &w, const int32_t *node, const Tracks &t, double step_max, int64_t n, double *step,
                              int32_t *next, cudaStream_t s);
cudaError_t launch_world_safety(const WorldTab &w, const int32_t *node, const Tracks &t, int64_t n, double *safety, cudaStream_t s);

// probes (vg_probe.cu)
cudaError_t probe_fp64_fma_rate(int launches, double *fma_per_s, cudaStream_t s);
cudaError_t probe_empty_launch(int launches, cudaStream_t s);
cudaError_t probe_stream(int q, const Tracks &t, int64_t n, void *out, bool vec, cudaStream_t s);

} // namespace vg
