// plic_kernels.cu -- kernels, launch logic and the C ABI of libplic (include/plic.h).
//
// One elementwise pass per call: 16 B read + 4 B written per cell, no reuse, so the kernels
// are built around HBM streaming, one float4 (4 cells) per array per thread per tile of 1024
// cells, 128-bit streaming stores.  None of the grids is persistent: one block per tile (or two),
// handed out by the hardware block scheduler ("Launch").  Three bodies:
//   map_tma      the HBM-bound kernels (analytic, SZ, Newton fast; plic_volume): a block owns two
//                consecutive tiles and brings their 8 input pieces into shared memory with 1-D bulk
//                asynchronous copies (cp.async.bulk, SASS UBLKCP) signalled on mbarriers, issued
//                all at once; 5 blocks resident per SM, so the bytes in flight per SM (160 KB) are
//                set by shared memory and not by registers x occupancy;
//   map_vec4     kernels bound by instruction issue (nested-fast, kawano): direct 128-bit
//                ld.global.nc.L1::no_allocate loads, one block per tile;
//   map_compact  the four precise methods (IEEE roots, libm trig, the paper's case order): every
//                cell takes the branch-free cheap part, the cells of the expensive cases (3)/(4)
//                and (1) are collected per tile in shared memory and evaluated by dense warps, so
//                that a warp never runs a case for a handful of its lanes.
// Not a contraction: no tensor cores.  Each byte is used exactly once by exactly one thread.
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <mutex>

#include "../../include/plic.h"
#include "plic_methods.cuh"
#include "plic_packed.cuh"
#include "plic_curvature.cuh"
#include "plic_probe.cuh"

#define PLIC_VERSION 106

namespace plic {

constexpr int kBlock = 256;        // threads per block
constexpr int kMaxDevices = 64;

__device__ __forceinline__ float4 ld_stream(const float4 *p) {
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                 : "l"(p));
    return v;
}
// the first input may be the output array (in-place call): no .nc on it
__device__ __forceinline__ float4 ld_stream_rw(const float4 *p) {
    float4 v;
    asm volatile("ld.global.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                 : "l"(p)
                 : "memory");
    return v;
}
__device__ __forceinline__ void st_stream(float4 *p, const float4 &v) {
    asm volatile("st.global.cs.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(v.x), "f"(v.y),
                 "f"(v.z), "f"(v.w)
                 : "memory");
}

// The body kernels are launched with programmatic stream serialization, so that on a stream of
// back-to-back calls the blocks of the next kernel become resident while the previous one drains
// and its launch latency is hidden.  Nothing is read from or written to global memory before
// this wait, which returns once the preceding kernel has completed and its writes are visible
// (a no-op after anything that is not a kernel).
__device__ __forceinline__ void grid_dependency_wait() {
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// op(V0-or-d0, nx, ny, nz) -> result, for one cell
enum : int { BODY_VEC4 = 0, BODY_TMA = 1, BODY_COMPACT = 2 };

template <int METHOD, bool FAST>
struct SolveOp {
    static constexpr int kMinBlocks = 0;      // resident blocks per SM asked of ptxas; 0 = its choice
    // the four precise methods run on map_compact, Listing 3 (kawano) on map_vec4
    static constexpr int kBody = METHOD == KAWANO ? BODY_VEC4 : BODY_COMPACT;
    static constexpr int kMethod = METHOD;
    static __device__ __forceinline__ float apply(float s, float x, float y, float z) {
        return solve_cell<METHOD, FAST>(s, x, y, z);
    }
    static __device__ __forceinline__ float4 apply4(const float4 &v, const float4 &a,
                                                    const float4 &b, const float4 &c) {
        return make_float4(apply(v.x, a.x, b.x, c.x), apply(v.y, a.y, b.y, c.y),
                           apply(v.z, a.z, b.z, c.z), apply(v.w, a.w, b.w, c.w));
    }
};
// The PLIC_FAST variants run on packed pairs (plic_packed.cuh); a single cell is a pair with
// both halves equal, so the scalar head/tail kernel gives bitwise the same result as the body.
template <int METHOD>
struct SolveOp<METHOD, true> {
    // nested intervals is bound by instruction issue and stays on map_vec4 at 6 blocks per SM
    // (40 registers); the other three are staged through shared memory (map_tma) at 5 blocks
    // per SM (48 registers, 5 x 32 KB of tiles)
    static constexpr int kBody = METHOD != NESTED ? BODY_TMA : BODY_VEC4;
    static constexpr int kMinBlocks = kBody == BODY_TMA ? 5 : 6;
    static __device__ __forceinline__ float apply(float s, float x, float y, float z) {
        return solve_pair_fast<METHOD>(F2{s, s}, F2{x, x}, F2{y, y}, F2{z, z}).x;
    }
    static __device__ __forceinline__ float4 apply4(const float4 &v, const float4 &a,
                                                    const float4 &b, const float4 &c) {
        const F2 lo = solve_pair_fast<METHOD>(F2{v.x, v.y}, F2{a.x, a.y}, F2{b.x, b.y}, F2{c.x, c.y});
        const F2 hi = solve_pair_fast<METHOD>(F2{v.z, v.w}, F2{a.z, a.w}, F2{b.z, b.w}, F2{c.z, c.w});
        return make_float4(lo.x, lo.y, hi.x, hi.y);
    }
};
// plic_volume also runs on packed pairs, branch-free, one division per cell (volume_pair).
struct VolumeOp {
    static constexpr int kBody = BODY_TMA;
    static constexpr int kMinBlocks = 5;
    static __device__ __forceinline__ float apply(float s, float x, float y, float z) {
        return volume_pair(F2{s, s}, F2{x, x}, F2{y, y}, F2{z, z}).x;
    }
    static __device__ __forceinline__ float4 apply4(const float4 &v, const float4 &a,
                                                    const float4 &b, const float4 &c) {
        const F2 lo = volume_pair(F2{v.x, v.y}, F2{a.x, a.y}, F2{b.x, b.y}, F2{c.x, c.y});
        const F2 hi = volume_pair(F2{v.z, v.w}, F2{a.z, a.w}, F2{b.z, b.w}, F2{c.z, c.w});
        return make_float4(lo.x, lo.y, hi.x, hi.y);
    }
};

// The "blank run" of eq. (33) as a map: d0 = V0 - 1/2, with the same four input streams and the
// same body kernel (map_tma) as the HBM-bound solvers, i.e. the ceiling of this access pattern
// (4 arrays read, 1 written) for bench.py's stream_ceiling.  The bulk copies bring all four
// tiles into shared memory whether or not the threads read them.
struct BlankOp {
    static constexpr int kBody = BODY_TMA;
    static constexpr int kMinBlocks = 5;
    static __device__ __forceinline__ float apply(float s, float, float, float) { return s - 0.5f; }
    static __device__ __forceinline__ float4 apply4(const float4 &v, const float4 &, const float4 &,
                                                    const float4 &) {
        return make_float4(v.x - 0.5f, v.y - 0.5f, v.z - 0.5f, v.w - 0.5f);
    }
};

// Body: n4 float4 groups (4 cells each), one block per tile of kBlock groups.  Not a persistent
// grid: with the tiles handed out by the hardware block scheduler the SMs that run faster (shorter
// memory latency, less divergent data) take more tiles; a grid-stride version of this kernel
// over SMs x resident blocks was 7-14 % slower (idle tail), 2-16 tiles per block 1-4 % slower.
constexpr int kVecTiles = 1;

template <class OP>
__global__ void __launch_bounds__(kBlock, OP::kMinBlocks)
map_vec4(const float4 *s, const float4 *__restrict__ nx, const float4 *__restrict__ ny,
         const float4 *__restrict__ nz, float4 *out, int64_t n4) {
    // s and out may be the same array (in-place call): no __restrict__, no .nc load on them
    grid_dependency_wait();
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i >= n4) return;
    const float4 v = ld_stream_rw(s + i);
    const float4 a = ld_stream(nx + i);
    const float4 b = ld_stream(ny + i);
    const float4 c = ld_stream(nz + i);
    st_stream(out + i, OP::apply4(v, a, b, c));
}

// ---------------------------------------------------------------------------------------
// map_tma: the same map with the input tiles brought into shared memory by the bulk-copy
// engine.  A tile is kBlock float4 groups (1024 cells) of each of the four arrays = 16 KB.  A
// block owns kTiles consecutive tiles: thread 0 arms one mbarrier per tile with the byte
// count and issues all 4 kTiles cp.async.bulk at once; every thread then waits for tile 0,
// copies its float4s to registers, computes and stores, then tile 1, ...  There is no stage
// reuse, hence no block barrier in the loop and no refill logic.  The grid is NOT persistent:
// one block per kTiles tiles, handed out by the hardware block scheduler, so SMs that see a
// shorter memory latency simply take more blocks -- a persistent grid-stride version of this
// kernel (3 stages, refilled) left 9 % of the SM time idle in its tail and was 5-14 % slower
// (DESIGN.md section 6).  Pipelining across tiles comes from the 5 resident blocks per SM
// being at different phases: 10 tiles = 160 KB in flight per SM.
// ---------------------------------------------------------------------------------------
constexpr int kTiles = 2;                                            // tiles per block
constexpr int kTileBytes = kBlock * 16;                              // one array's tile
constexpr int kTmaSmem = kTiles * 4 * kTileBytes + kTiles * 8;       // tiles + mbarriers

__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ bool elect_one() {                        // one lane of the (converged) warp
    unsigned pred;
    asm volatile("{ .reg .pred p; elect.sync _|p, 0xffffffff; selp.u32 %0, 1, 0, p; }" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

template <class OP>
__global__ void __launch_bounds__(kBlock, OP::kMinBlocks)
map_tma(const float4 *s, const float4 *__restrict__ nx, const float4 *__restrict__ ny,
        const float4 *__restrict__ nz, float4 *out, int64_t n4) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4 *buf = reinterpret_cast<float4 *>(smem_raw);              // [kTiles][4][kBlock]
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + kTiles * 4 * kTileBytes);
    const int tid = threadIdx.x;
    const int64_t ntiles = (n4 + kBlock - 1) / kBlock;
    const int64_t first = (int64_t)blockIdx.x * kTiles;
    // one elected lane of warp 0 issues the copies; the warp index is broadcast so that the branch is
    // provably warp-uniform (the bulk-copy instructions run on the uniform datapath: under a
    // divergent branch ptxas wraps each of them in an election loop)
    const bool issuer = __shfl_sync(0xffffffffu, tid >> 5, 0) == 0 && elect_one();
    if (issuer) {
        for (int k = 0; k < kTiles; ++k) mbar_init(&full[k], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        grid_dependency_wait();                     // before the first read of global memory
#pragma unroll
        for (int k = 0; k < kTiles; ++k) {
            const int64_t tile = first + k;
            if (tile < ntiles) {
                const int64_t base = tile * kBlock;
                const int64_t rem = n4 - base;
                const uint32_t bytes = (uint32_t)(rem < kBlock ? rem : kBlock) * 16u;   // ragged last tile
                float4 *dst = buf + k * 4 * kBlock;
                mbar_expect_tx(&full[k], 4 * bytes);
                bulk_g2s(dst, s + base, bytes, &full[k]);
                bulk_g2s(dst + kBlock, nx + base, bytes, &full[k]);
                bulk_g2s(dst + 2 * kBlock, ny + base, bytes, &full[k]);
                bulk_g2s(dst + 3 * kBlock, nz + base, bytes, &full[k]);
            }
        }
    }
    __syncthreads();                                                 // barriers initialised
#pragma unroll
    for (int k = 0; k < kTiles; ++k) {
        const int64_t tile = first + k;
        if (tile >= ntiles) break;
        mbar_wait(&full[k], 0);
        const float4 *src = buf + k * 4 * kBlock;
        // in a ragged last tile the slots past the end were never written: they are computed
        // and dropped, never stored
        const float4 v = src[tid], a = src[kBlock + tid], b = src[2 * kBlock + tid],
                     c = src[3 * kBlock + tid];
        const int64_t i = tile * kBlock + tid;
        if (i < n4) st_stream(out + i, OP::apply4(v, a, b, c));
    }
}

// ---------------------------------------------------------------------------------------
// map_compact: the precise methods with the expensive cases compacted per tile.
//
// The precise methods keep IEEE roots and libm cbrt / asin / sin / acos / cos, whose cost
// (60-110 instructions) is only due for the cells of cases (3)/(4) (38 % of random cells) and
// (1) (6 %).  With a branch per cell a warp pays for every case any of its lanes is in: 10-15
// of 32 lanes were active per issued instruction and the kernels ran 1.7-2.4x slower on mixed
// than on case-sorted cells.  Here a block of 256 threads owns one tile of 1024 cells:
//   phase 1  every thread reduces its 4 cells (eq. (2)-(5)), evaluates Precise<M>::cheap() --
//            cases (5) and (2) and the case decision, no branch -- writes the 4 offsets to
//            `dres`, the reduced cells (n1, n2, n3, V) to `cells`, and appends the slots of its
//            heavy cells to a queue in shared memory: cases (3)/(4) from the front, case (1)
//            from the back (one packed shared atomic per warp after a warp scan of the packed
//            counts);
//   phase 2  the queue is evaluated by whole warps: entry j by thread j mod 256, the case-(1)
//            entries starting at a warp boundary, so every warp runs one case with all its
//            lanes (but the last of each kind), and the results overwrite their `dres` slots;
//   phase 3  every thread reads its 4 offsets back, restores the sign (eq. (8)) and stores.
// The arithmetic per cell is that of Solver<M, false>::reduced_offset(), bitwise.
// ---------------------------------------------------------------------------------------
constexpr int kTileCells = 4 * kBlock;

template <int METHOD>
__global__ void __launch_bounds__(kBlock, 5)
map_compact(const float4 *s, const float4 *__restrict__ nx, const float4 *__restrict__ ny,
            const float4 *__restrict__ nz, float4 *out, int64_t n4) {
    __shared__ float4 cells[kTileCells];             // (n1, n2, n3, V) of every cell of the tile
    __shared__ __align__(16) float dres[kTileCells]; // reduced offset d of every cell of the tile
    __shared__ unsigned short queue[kTileCells];     // cell slots: heavy-A from the front, heavy-B from the back
    __shared__ unsigned count;                       // heavy-A entries | heavy-B entries << 16
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    if (tid == 0) count = 0;
    __syncthreads();
    grid_dependency_wait();
    const int64_t i = (int64_t)blockIdx.x * kBlock + tid;
    const bool live = i < n4;
    // threads past the end carry n = (0, 0, 1), V0 = 0: case (5) in every method (n1 + n2 = 0 <= 2 V n3 = 0),
    // nothing queued.  (The zero normal would not do: SZ divides by S = 0 and its NaN fails every case
    // test, which queues the dead slots as heavy cells.)
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f), a = v, b = v, c = make_float4(1.f, 1.f, 1.f, 1.f);
    if (live) {
        v = ld_stream_rw(s + i);
        a = ld_stream(nx + i);
        b = ld_stream(ny + i);
        c = ld_stream(nz + i);
    }
    const float V0[4] = {v.x, v.y, v.z, v.w};
    const float X[4] = {a.x, a.y, a.z, a.w}, Y[4] = {b.x, b.y, b.z, b.w}, Z[4] = {c.x, c.y, c.z, c.w};
    float d[4], hS[4];
    int kind[4];
    unsigned mine = 0;                               // packed counts of this thread
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const Reduced cell = reduce_cell(V0[k], X[k], Y[k], Z[k]);
        hS[k] = half_l1(cell);
        d[k] = Precise<METHOD>::cheap(cell.n1, cell.n2, cell.n3, cell.V, kind[k]);
        mine += (unsigned)kind[k];
        cells[4 * tid + k] = make_float4(cell.n1, cell.n2, cell.n3, cell.V);
    }
    reinterpret_cast<float4 *>(dres)[tid] = make_float4(d[0], d[1], d[2], d[3]);
    unsigned scan = mine;                            // inclusive warp scan of both counts at once
#pragma unroll
    for (int o = 1; o < 32; o <<= 1)                 // the shuffle's predicate is "source lane in range"
        asm("{ .reg .pred p; .reg .u32 t; shfl.sync.up.b32 t|p, %0, %1, 0, 0xffffffff; @p add.u32 %0, %0, t; }"
            : "+r"(scan)
            : "r"(o));
    unsigned pos = 0;
    if (lane == 31) pos = atomicAdd(&count, scan);
    pos = __shfl_sync(0xffffffffu, pos, 31) + scan - mine;       // packed queue positions of this thread
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const unsigned idx = kind[k] == KIND_HEAVY_A ? (pos & 0xffffu) : (unsigned)(kTileCells - 1) - (pos >> 16);
        if (kind[k] != KIND_DONE) queue[idx] = (unsigned short)(4 * tid + k);
        pos += (unsigned)kind[k];
    }
    __syncthreads();
    const unsigned na = count & 0xffffu, nb = count >> 16;
    const unsigned na32 = (na + 31u) & ~31u;         // case-(1) entries start at a warp boundary
    for (unsigned j = tid; j < na32 + nb; j += kBlock) {
        if (j < na32) {
            if (j < na) {
                const unsigned slot = queue[j];
                const float4 e = cells[slot];
                dres[slot] = Precise<METHOD>::heavy_a(e.x, e.y, e.z, e.w);
            }
        } else {
            const unsigned slot = queue[(unsigned)(kTileCells - 1) - (j - na32)];
            const float4 e = cells[slot];
            dres[slot] = Precise<METHOD>::heavy_b(e.x, e.y, e.z, e.w);
        }
    }
    __syncthreads();
    if (!live) return;
    const float4 r = reinterpret_cast<const float4 *>(dres)[tid];
    st_stream(out + i, make_float4(restore_cell<true>(V0[0], hS[0], r.x), restore_cell<true>(V0[1], hS[1], r.y),
                                   restore_cell<true>(V0[2], hS[2], r.z), restore_cell<true>(V0[3], hS[3], r.w)));
}

// Scalar: cells [0, head) and [tail0, N) (head/tail of the vector body), or the whole
// range when the five pointers do not share an alignment (head = N).
template <class OP>
__global__ void __launch_bounds__(kBlock)
map_scalar(const float *s, const float *__restrict__ nx, const float *__restrict__ ny,
           const float *__restrict__ nz, float *out, int64_t head, int64_t tail0, int64_t N) {
    const int64_t stride = (int64_t)gridDim.x * kBlock;
    const int64_t count = head + (N - tail0);
    for (int64_t j = (int64_t)blockIdx.x * kBlock + threadIdx.x; j < count; j += stride) {
        const int64_t i = j < head ? j : tail0 + (j - head);
        out[i] = OP::apply(s[i], nx[i], ny[i], nz[i]);
    }
}

// ---------------------------------------------------------------------------------------
// launch geometry: one block per tile (map_vec4, map_compact) or per kTiles tiles (map_tma)
// ---------------------------------------------------------------------------------------
struct DeviceInfo {
    std::once_flag once;
    int sms = 0;
    cudaError_t err = cudaSuccess;
};
static DeviceInfo g_dev[kMaxDevices];
static std::atomic<int64_t> g_launches{0};

typedef void (*vec_kernel_t)(const float4 *, const float4 *, const float4 *, const float4 *,
                             float4 *, int64_t);
typedef void (*scalar_kernel_t)(const float *, const float *, const float *, const float *,
                                float *, int64_t, int64_t, int64_t);

// body kernel of an op, the dynamic shared memory it needs and the tiles one block takes
struct BodyKernel {
    vec_kernel_t fn;
    int smem;
    int tiles;
};
template <class OP>
static BodyKernel body_of() {
    if constexpr (OP::kBody == BODY_TMA)
        return BodyKernel{map_tma<OP>, kTmaSmem, kTiles};
    else if constexpr (OP::kBody == BODY_COMPACT)
        return BodyKernel{map_compact<OP::kMethod>, 0, 1};
    else
        return BodyKernel{map_vec4<OP>, 0, kVecTiles};
}
static BodyKernel vec_kernel(int k) {
    switch (k) {
        case 0: return body_of<SolveOp<ANALYTIC, false>>();
        case 1: return body_of<SolveOp<SZ, false>>();
        case 2: return body_of<SolveOp<NEWTON, false>>();
        case 3: return body_of<SolveOp<NESTED, false>>();
        case 4: return body_of<SolveOp<ANALYTIC, true>>();
        case 5: return body_of<SolveOp<SZ, true>>();
        case 6: return body_of<SolveOp<NEWTON, true>>();
        case 7: return body_of<SolveOp<NESTED, true>>();
        case 9: return body_of<SolveOp<KAWANO, false>>();
        case 10: return body_of<BlankOp>();
        default: return body_of<VolumeOp>();
    }
}
static scalar_kernel_t scalar_kernel(int k) {
    switch (k) {
        case 0: return map_scalar<SolveOp<ANALYTIC, false>>;
        case 1: return map_scalar<SolveOp<SZ, false>>;
        case 2: return map_scalar<SolveOp<NEWTON, false>>;
        case 3: return map_scalar<SolveOp<NESTED, false>>;
        case 4: return map_scalar<SolveOp<ANALYTIC, true>>;
        case 5: return map_scalar<SolveOp<SZ, true>>;
        case 6: return map_scalar<SolveOp<NEWTON, true>>;
        case 7: return map_scalar<SolveOp<NESTED, true>>;
        case 9: return map_scalar<SolveOp<KAWANO, false>>;
        case 10: return map_scalar<BlankOp>;
        default: return map_scalar<VolumeOp>;
    }
}

// kernel index for a method id; -1 if the id is unknown
static int kernel_index(int method) {
    if (method == PLIC_METHOD_KAWANO) return 2 * PLIC_NUM_METHODS + 1;     // precise only
    if (method == PLIC_METHOD_BLANK) return 2 * PLIC_NUM_METHODS + 2;      // d0 = V0 - 1/2
    const int base = method & ~PLIC_FAST;
    if (base < 0 || base >= PLIC_NUM_METHODS) return -1;
    return base + ((method & PLIC_FAST) ? PLIC_NUM_METHODS : 0);
}
constexpr int kVolumeKernel = 2 * PLIC_NUM_METHODS;

static DeviceInfo *device_info(cudaError_t *err) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
        *err = e != cudaSuccess ? e : cudaErrorInvalidDevice;
        return nullptr;
    }
    DeviceInfo *info = &g_dev[dev];
    std::call_once(info->once, [info, dev]() {
        info->err = cudaDeviceGetAttribute(&info->sms, cudaDevAttrMultiProcessorCount, dev);
    });
    *err = info->err;
    return info->err == cudaSuccess ? info : nullptr;
}

// blocks for `units` work items (float4 groups or cells) at kBlock per tile and `per` tiles per block
static int grid_for(int64_t units, int per) {
    const int64_t tiles = (units + kBlock - 1) / kBlock;
    const int64_t blocks = (tiles + per - 1) / per;
    return (int)(blocks < 1 ? 1 : (blocks > 0x7fffffffLL ? 0x7fffffffLL : blocks));
}
static_assert(kTmaSmem <= 48 * 1024, "map_tma fits the default dynamic shared memory limit");

static int launch_map(int k, const float *s, const float *nx, const float *ny, const float *nz,
                      float *out, int64_t N, cudaStream_t stream) {
    if (N < 0) return PLIC_ERR_SIZE;
    if (N == 0) return PLIC_OK;
    if (!s || !nx || !ny || !nz || !out) return PLIC_ERR_NULL;
    const uintptr_t ps[5] = {(uintptr_t)s, (uintptr_t)nx, (uintptr_t)ny, (uintptr_t)nz,
                             (uintptr_t)out};
    bool same = true;
    for (int i = 0; i < 5; ++i) {
        if (ps[i] & 3u) return PLIC_ERR_ALIGN;
        if ((ps[i] & 15u) != (ps[0] & 15u)) same = false;
    }
    // cells before the first 16-byte boundary, then n4 full float4 groups, then the tail
    int64_t head = same ? (int64_t)(((16u - (ps[0] & 15u)) & 15u) >> 2) : N;
    if (head > N) head = N;
    const int64_t n4 = (N - head) / 4;
    const int64_t tail0 = head + 4 * n4;

    if (n4 > 0) {
        const BodyKernel body = vec_kernel(k);
        const int per = body.tiles;
        if ((n4 + kBlock - 1) / kBlock > (int64_t)per * 0x7fffffffLL) return PLIC_ERR_SIZE;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)grid_for(n4, per));
        cfg.blockDim = dim3(kBlock);
        cfg.dynamicSmemBytes = (size_t)body.smem;
        cfg.stream = stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        if (cudaLaunchKernelEx(&cfg, body.fn, (const float4 *)(s + head), (const float4 *)(nx + head),
                               (const float4 *)(ny + head), (const float4 *)(nz + head),
                               (float4 *)(out + head), n4) != cudaSuccess)
            return PLIC_ERR_LAUNCH;
        g_launches.fetch_add(1, std::memory_order_relaxed);
    }
    const int64_t rest = head + (N - tail0);
    if (rest > 0) {
        scalar_kernel(k)<<<grid_for(rest, 1), kBlock, 0, stream>>>(s, nx, ny, nz, out, head,
                                                                      tail0, N);
        g_launches.fetch_add(1, std::memory_order_relaxed);
    }
    return cudaPeekAtLastError() == cudaSuccess ? PLIC_OK : PLIC_ERR_LAUNCH;
}

// ---------------------------------------------------------------------------------------
// roundtrip_kernel: the paper's benchmark loop (sect. 2.6, eq. (31)-(33)).  One thread per
// normal; L volumes in series, two per step on a packed pair (V0_l, V0_{l+1}) that shares
// the normal, so everything that depends on n alone is hoisted out of the loop by the
// compiler -- the same situation as the paper's OpenCL kernel.
// METHOD = -1 is the blank run of eq. (33).
// ---------------------------------------------------------------------------------------
template <int METHOD, bool FAST>
struct PairOffset {                                   // precise kernels: two scalar solves
    static __device__ __forceinline__ F2 d0(F2 V0, F2 x, F2 y, F2 z) {
        return F2{solve_cell<METHOD, false>(V0.x, x.x, y.x, z.x),
                  solve_cell<METHOD, false>(V0.y, x.y, y.y, z.y)};
    }
};
template <int METHOD>
struct PairOffset<METHOD, true> {
    static __device__ __forceinline__ F2 d0(F2 V0, F2 x, F2 y, F2 z) {
        return solve_pair_fast<METHOD>(V0, x, y, z);
    }
};
template <>
struct PairOffset<-1, true> {
    static __device__ __forceinline__ F2 d0(F2 V0, F2, F2, F2) { return add2(V0, f2(-0.5f)); }
};

template <int METHOD, bool FAST>
__global__ void __launch_bounds__(kBlock)
roundtrip_kernel(const float *__restrict__ nx, const float *__restrict__ ny,
                 const float *__restrict__ nz, float *__restrict__ E, int64_t N, int L) {
    const float h = 1.0f / (float)(L - 1);
    const int64_t stride = (int64_t)gridDim.x * kBlock;
    for (int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x; i < N; i += stride) {
        const float x = nx[i], y = ny[i], z = nz[i];
        const F2 X{x, x}, Y{y, y}, Z{z, z};
        F2 acc{0.0f, 0.0f};
        for (int l = 0; l < L; l += 2) {
            // V0_l = l / (L - 1); the last one is exactly 1.  For odd L the second half of the
            // last pair is a repeat of V0 = 1 and is not accumulated.
            const F2 V0{l >= L - 1 ? 1.0f : (float)l * h, l + 1 >= L - 1 ? 1.0f : (float)(l + 1) * h};
            const F2 d0 = PairOffset<METHOD, FAST>::d0(V0, X, Y, Z);
            const F2 V = volume_pair(d0, X, Y, Z);
            F2 err = abs2(sub2(V, V0));                                         // eq. (31)
            if (METHOD == KAWANO) {          // Listing 3's NaN propagates into the average;
                if (d0.x != d0.x) err.x = d0.x;   // volume_pair itself never returns NaN
                if (d0.y != d0.y) err.y = d0.y;
            }
            acc.x += err.x;
            if (l + 1 < L) acc.y += err.y;
        }
        E[i] = (acc.x + acc.y) / (float)L;
    }
}

typedef void (*roundtrip_kernel_t)(const float *, const float *, const float *, float *, int64_t,
                                   int);
static roundtrip_kernel_t roundtrip_kernel_of(int k) {
    switch (k) {
        case 0: return roundtrip_kernel<ANALYTIC, false>;
        case 1: return roundtrip_kernel<SZ, false>;
        case 2: return roundtrip_kernel<NEWTON, false>;
        case 3: return roundtrip_kernel<NESTED, false>;
        case 4: return roundtrip_kernel<ANALYTIC, true>;
        case 5: return roundtrip_kernel<SZ, true>;
        case 6: return roundtrip_kernel<NEWTON, true>;
        case 7: return roundtrip_kernel<NESTED, true>;
        case 9: return roundtrip_kernel<KAWANO, false>;
        default: return roundtrip_kernel<-1, true>;
    }
}

// ---------------------------------------------------------------------------------------
// plane-sphere maps (sect. 3): one array in, one array out, 8 B per cell.  map1_vec4 handles
// the 16-byte aligned body, map1_scalar head, tail and misaligned ranges.
// ---------------------------------------------------------------------------------------
struct SphereSolveFastOp {
    static __device__ __forceinline__ F2 apply2(F2 v) { return sphere_solve_pair_fast(v); }
};
struct SphereSolveOp {
    static __device__ __forceinline__ F2 apply2(F2 v) {
        return F2{sphere_solve_cell(v.x), sphere_solve_cell(v.y)};
    }
};
struct SphereVolumeOp {
    static __device__ __forceinline__ F2 apply2(F2 v) { return sphere_volume_pair(v); }
};

template <class OP>
__global__ void __launch_bounds__(kBlock, 8)
map1_vec4(const float4 *__restrict__ in, float4 *__restrict__ out, int64_t n4) {
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;      // one block per tile, as map_vec4
    if (i >= n4) return;
    const float4 v = ld_stream(in + i);
    const F2 lo = OP::apply2(F2{v.x, v.y}), hi = OP::apply2(F2{v.z, v.w});
    st_stream(out + i, make_float4(lo.x, lo.y, hi.x, hi.y));
}
template <class OP>
__global__ void __launch_bounds__(kBlock)
map1_scalar(const float *__restrict__ in, float *__restrict__ out, int64_t head, int64_t tail0,
            int64_t N) {
    const int64_t stride = (int64_t)gridDim.x * kBlock;
    const int64_t count = head + (N - tail0);
    for (int64_t j = (int64_t)blockIdx.x * kBlock + threadIdx.x; j < count; j += stride) {
        const int64_t i = j < head ? j : tail0 + (j - head);
        const float v = in[i];
        out[i] = OP::apply2(F2{v, v}).x;
    }
}

template <class OP>
static int launch_map1(const float *in, float *out, int64_t N, cudaStream_t stream) {
    if (N < 0) return PLIC_ERR_SIZE;
    if (N == 0) return PLIC_OK;
    if (!in || !out) return PLIC_ERR_NULL;
    const uintptr_t pi = (uintptr_t)in, po = (uintptr_t)out;
    if ((pi | po) & 3u) return PLIC_ERR_ALIGN;
    cudaError_t err;
    const DeviceInfo *info = device_info(&err);
    if (!info) return PLIC_ERR_LAUNCH;
    int64_t head = (pi & 15u) == (po & 15u) ? (int64_t)(((16u - (pi & 15u)) & 15u) >> 2) : N;
    if (head > N) head = N;
    const int64_t n4 = (N - head) / 4;
    const int64_t tail0 = head + 4 * n4;
    const int64_t full = (int64_t)info->sms * 8;                     // 8 resident blocks of 256
    if (n4 > 0) {
        const int64_t need = (n4 + kBlock - 1) / kBlock;
        if (need > 0x7fffffffLL) return PLIC_ERR_SIZE;
        map1_vec4<OP><<<(int)need, kBlock, 0, stream>>>(
            (const float4 *)(in + head), (float4 *)(out + head), n4);
        g_launches.fetch_add(1, std::memory_order_relaxed);
    }
    const int64_t rest = head + (N - tail0);
    if (rest > 0) {
        const int64_t need = (rest + kBlock - 1) / kBlock;
        map1_scalar<OP><<<(int)(need < full ? need : full), kBlock, 0, stream>>>(in, out, head,
                                                                                 tail0, N);
        g_launches.fetch_add(1, std::memory_order_relaxed);
    }
    return cudaPeekAtLastError() == cudaSuccess ? PLIC_OK : PLIC_ERR_LAUNCH;
}

// ---------------------------------------------------------------------------------------
// host-array API: chunked, three-stage pipeline (H2D | kernel | D2H) over three streams
// ---------------------------------------------------------------------------------------
constexpr int kSlots = 3;
constexpr int64_t kChunk = (int64_t)1 << 22;     // cells per chunk: 64 MiB in, 16 MiB out

struct HostPipe {
    bool ready = false;
    cudaStream_t stream[kSlots] = {nullptr, nullptr, nullptr};
    float *buf[kSlots] = {nullptr, nullptr, nullptr};     // 5 * kChunk floats each
};
static HostPipe g_pipe[kMaxDevices];
static std::mutex g_pipe_mutex;

static void pipe_free(HostPipe *p) {
    for (int i = 0; i < kSlots; ++i) {
        if (p->buf[i]) cudaFree(p->buf[i]);
        if (p->stream[i]) cudaStreamDestroy(p->stream[i]);
        p->buf[i] = nullptr;
        p->stream[i] = nullptr;
    }
    p->ready = false;
}

static bool pipe_init(HostPipe *p) {
    if (p->ready) return true;
    for (int i = 0; i < kSlots; ++i) {
        if (cudaStreamCreateWithFlags(&p->stream[i], cudaStreamNonBlocking) != cudaSuccess ||
            cudaMalloc((void **)&p->buf[i], 5 * kChunk * sizeof(float)) != cudaSuccess) {
            pipe_free(p);
            cudaGetLastError();
            return false;
        }
    }
    p->ready = true;
    return true;
}

static int host_map(int k, const float *s, const float *nx, const float *ny, const float *nz,
                    float *out, int64_t N) {
    if (N < 0) return PLIC_ERR_SIZE;
    if (N == 0) return PLIC_OK;
    if (!s || !nx || !ny || !nz || !out) return PLIC_ERR_NULL;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return PLIC_ERR_LAUNCH;
    std::lock_guard<std::mutex> lock(g_pipe_mutex);
    HostPipe *p = &g_pipe[dev];
    if (!pipe_init(p)) return PLIC_ERR_LAUNCH;
    const float *in[4] = {s, nx, ny, nz};
    int rc = PLIC_OK;
    int slot = 0;
    for (int64_t off = 0; off < N && rc == PLIC_OK; off += kChunk, slot = (slot + 1) % kSlots) {
        const int64_t n = (N - off) < kChunk ? (N - off) : kChunk;
        cudaStream_t st = p->stream[slot];     // stream order makes the slot's reuse safe
        float *b = p->buf[slot];
        for (int a = 0; a < 4; ++a)
            if (cudaMemcpyAsync(b + a * kChunk, in[a] + off, n * sizeof(float),
                                cudaMemcpyHostToDevice, st) != cudaSuccess)
                rc = PLIC_ERR_LAUNCH;
        if (rc == PLIC_OK)
            rc = launch_map(k, b, b + kChunk, b + 2 * kChunk, b + 3 * kChunk, b + 4 * kChunk, n, st);
        if (rc == PLIC_OK &&
            cudaMemcpyAsync(out + off, b + 4 * kChunk, n * sizeof(float), cudaMemcpyDeviceToHost,
                            st) != cudaSuccess)
            rc = PLIC_ERR_LAUNCH;
    }
    for (int i = 0; i < kSlots; ++i)
        if (cudaStreamSynchronize(p->stream[i]) != cudaSuccess) rc = PLIC_ERR_LAUNCH;
    if (rc != PLIC_OK) cudaGetLastError();
    return rc;
}

}  // namespace plic

#include "plic_storage.cuh"       // binary16-storage and fp64 variants (uses the kernels and helpers above)

// ---------------------------------------------------------------------------------------
// C ABI
// ---------------------------------------------------------------------------------------
extern "C" {

int plic_solve(const float *V0, const float *nx, const float *ny, const float *nz, float *d0,
               int64_t N, int method, cudaStream_t stream) {
    const int k = plic::kernel_index(method);
    if (k < 0) return PLIC_ERR_METHOD;
    return plic::launch_map(k, V0, nx, ny, nz, d0, N, stream);
}

int plic_volume(const float *d0, const float *nx, const float *ny, const float *nz, float *V0,
                int64_t N, cudaStream_t stream) {
    return plic::launch_map(plic::kVolumeKernel, d0, nx, ny, nz, V0, N, stream);
}

int plic_solve_h(const uint16_t *V0, const uint16_t *nx, const uint16_t *ny, const uint16_t *nz,
                 uint16_t *d0, float *d0_f32, int64_t N, int method, cudaStream_t stream) {
    const int k = plic::kernel_index(method);
    if (k < 0) return PLIC_ERR_METHOD;
    return plic::launch_map_io(plic::io_kernel_h(k), 2, V0, nx, ny, nz, d0, d0_f32, N, stream);
}

int plic_volume_h(const uint16_t *d0, const uint16_t *nx, const uint16_t *ny, const uint16_t *nz,
                  uint16_t *V0, float *V0_f32, int64_t N, cudaStream_t stream) {
    return plic::launch_map_io(plic::io_kernel_h(plic::kVolumeKernel), 2, d0, nx, ny, nz, V0, V0_f32, N, stream);
}

int plic_solve_f64(const double *V0, const double *nx, const double *ny, const double *nz, double *d0,
                   int64_t N, int method, cudaStream_t stream) {
    const int k = plic::kernel_index(method);
    if (k < 0) return PLIC_ERR_METHOD;
    return plic::launch_map_io(plic::io_kernel_d(k), 8, V0, nx, ny, nz, d0, nullptr, N, stream);
}

int plic_roundtrip_error(const float *nx, const float *ny, const float *nz, float *E, int64_t N,
                         int L, int method, cudaStream_t stream) {
    const int k = method == PLIC_METHOD_BLANK ? plic::kVolumeKernel : plic::kernel_index(method);   // blank: default case
    if (k < 0) return PLIC_ERR_METHOD;
    if (N < 0 || L < 2) return PLIC_ERR_SIZE;
    if (N == 0) return PLIC_OK;
    if (!nx || !ny || !nz || !E) return PLIC_ERR_NULL;
    if (((uintptr_t)nx | (uintptr_t)ny | (uintptr_t)nz | (uintptr_t)E) & 3u) return PLIC_ERR_ALIGN;
    // compute bound: one thread per normal, one block per 256 normals (hardware block scheduling)
    plic::roundtrip_kernel_of(k)<<<plic::grid_for(N, 1), plic::kBlock, 0, stream>>>(
        nx, ny, nz, E, N, L);
    plic::g_launches.fetch_add(1, std::memory_order_relaxed);
    return cudaPeekAtLastError() == cudaSuccess ? PLIC_OK : PLIC_ERR_LAUNCH;
}

int plic_sphere_solve(const float *V0, float *d0, int64_t N, int fast, cudaStream_t stream) {
    if (fast != 0 && fast != PLIC_FAST) return PLIC_ERR_METHOD;
    return fast ? plic::launch_map1<plic::SphereSolveFastOp>(V0, d0, N, stream)
                : plic::launch_map1<plic::SphereSolveOp>(V0, d0, N, stream);
}

int plic_sphere_volume(const float *d0, float *V0, int64_t N, cudaStream_t stream) {
    return plic::launch_map1<plic::SphereVolumeOp>(d0, V0, N, stream);
}

int plic_curvature(const float *phi, float *kappa, int nx, int ny, int nz, int32_t *work,
                   int64_t work_entries, cudaStream_t stream) {
    if (nx < 0 || ny < 0 || nz < 0) return PLIC_ERR_SIZE;
    const int64_t ncells = (int64_t)nx * ny * nz;
    if (ncells > 0x7fffffffLL) return PLIC_ERR_SIZE;
    if (ncells == 0) return PLIC_OK;
    if (!phi || !kappa || !work) return PLIC_ERR_NULL;
    if (work_entries < 2) return PLIC_ERR_SIZE;
    if (((uintptr_t)phi | (uintptr_t)kappa | (uintptr_t)work) & 3u) return PLIC_ERR_ALIGN;
    cudaError_t err;
    const plic::DeviceInfo *info = plic::device_info(&err);
    if (!info) return PLIC_ERR_LAUNCH;
    int64_t cap64 = work_entries - 1;
    if (cap64 > ncells) cap64 = ncells;
    const int capacity = (int)cap64;
    // three launches, each a programmatic dependent launch of its predecessor: the launch latencies
    // hide behind the preceding kernel's tail; every kernel waits (griddepcontrol.wait) before its
    // first global access
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    cfg.gridDim = dim3(1);
    cfg.blockDim = dim3(32);
    if (cudaLaunchKernelEx(&cfg, plic::curv_reset, (int *)work) != cudaSuccess) return PLIC_ERR_LAUNCH;
    int64_t need, full = (int64_t)info->sms * 8;
    cfg.blockDim = dim3(256);
    if ((((uintptr_t)phi | (uintptr_t)kappa) & 15u) == 0 && ncells >= 4) {
        need = (ncells / 4 + 256 * plic::kMarkGroups - 1) / (256 * plic::kMarkGroups);
        cfg.gridDim = dim3((unsigned)need);
        if (cudaLaunchKernelEx(&cfg, plic::curv_mark4, (const float4 *)phi, (float4 *)kappa, nx, ny, nz,
                               (int *)work, capacity) != cudaSuccess)
            return PLIC_ERR_LAUNCH;
    } else {
        need = (ncells + 255) / 256;
        cfg.gridDim = dim3((unsigned)(need < full ? need : full));
        if (cudaLaunchKernelEx(&cfg, plic::curv_mark, phi, kappa, nx, ny, nz, (int *)work, capacity) !=
            cudaSuccess)
            return PLIC_ERR_LAUNCH;
    }
    need = ((int64_t)capacity * plic::kPointLanes + plic::kCurvBlock - 1) / plic::kCurvBlock;
    full = (int64_t)info->sms * 16;
    cfg.gridDim = dim3((unsigned)(need < full ? need : full));
    cfg.blockDim = dim3(plic::kCurvBlock);
    const int *list = work;
    if (cudaLaunchKernelEx(&cfg, plic::curv_cells, phi, kappa, nx, ny, list, capacity) != cudaSuccess)
        return PLIC_ERR_LAUNCH;
    plic::g_launches.fetch_add(3, std::memory_order_relaxed);
    return cudaPeekAtLastError() == cudaSuccess ? PLIC_OK : PLIC_ERR_LAUNCH;
}

int plic_solve_host(const float *V0, const float *nx, const float *ny, const float *nz,
                    float *d0, int64_t N, int method) {
    const int k = plic::kernel_index(method);
    if (k < 0) return PLIC_ERR_METHOD;
    return plic::host_map(k, V0, nx, ny, nz, d0, N);
}

int plic_volume_host(const float *d0, const float *nx, const float *ny, const float *nz,
                     float *V0, int64_t N) {
    return plic::host_map(plic::kVolumeKernel, d0, nx, ny, nz, V0, N);
}

void plic_host_release(void) {
    std::lock_guard<std::mutex> lock(plic::g_pipe_mutex);
    int cur = 0;
    const bool have = cudaGetDevice(&cur) == cudaSuccess;
    for (int d = 0; d < plic::kMaxDevices; ++d) {
        if (!plic::g_pipe[d].ready) continue;
        cudaSetDevice(d);
        plic::pipe_free(&plic::g_pipe[d]);
    }
    if (have) cudaSetDevice(cur);
}

const char *plic_method_name(int method) {
    static const char *names[2 * PLIC_NUM_METHODS] = {
        "analytic",      "sz",      "newton",      "nested",
        "analytic-fast", "sz-fast", "newton-fast", "nested-fast"};
    if (method == PLIC_METHOD_BLANK) return "blank";
    if (method == PLIC_METHOD_KAWANO) return "kawano";
    const int k = plic::kernel_index(method);
    return k < 0 ? nullptr : names[k];
}

const char *plic_error_string(int code) {
    switch (code) {
        case PLIC_OK: return "ok";
        case PLIC_ERR_NULL: return "null pointer with N > 0";
        case PLIC_ERR_SIZE: return "size argument out of range";
        case PLIC_ERR_METHOD: return "unknown method id";
        case PLIC_ERR_LAUNCH: return "CUDA runtime error";
        case PLIC_ERR_ALIGN: return "pointer not aligned to its element size";
        case PLIC_ERR_CAPACITY:
            return "lattice has more interior cells than plic_curvature_static's built-in list holds "
                   "(PLIC_CURVATURE_STATIC_MAX_POINTS); use plic_curvature with your own work array";
        default: return "unknown error code";
    }
}

int plic_version(void) { return PLIC_VERSION; }

int plic_pipe_probe(int pipe, int trips, float *sink, int64_t *warp_instructions, cudaStream_t stream) {
    if (pipe < 0 || pipe >= plic::PROBE_COUNT) return PLIC_ERR_METHOD;
    if (trips < 0) return PLIC_ERR_SIZE;
    if (!sink || !warp_instructions) return PLIC_ERR_NULL;
    cudaError_t err;
    const plic::DeviceInfo *info = plic::device_info(&err);
    if (!info) return PLIC_ERR_LAUNCH;
    const int grid = info->sms * plic::kProbeBlocksPerSm;
    const int64_t warps = (int64_t)grid * (plic::kBlock / 32);
    int64_t per_trip = 0;
#define PLIC_PROBE_CASE(P) \
    case plic::P: plic::pipe_probe<plic::P><<<grid, plic::kBlock, 0, stream>>>(sink, trips); \
                  per_trip = (int64_t)plic::kProbeChains * plic::kProbeUnroll * plic::ProbeOp<plic::P>::kInst; break;
    switch (pipe) {
        PLIC_PROBE_CASE(PROBE_FFMA)
        PLIC_PROBE_CASE(PROBE_FFMA2)
        PLIC_PROBE_CASE(PROBE_MUFU)
        PLIC_PROBE_CASE(PROBE_FMNMX)
        PLIC_PROBE_CASE(PROBE_LOP3)
        PLIC_PROBE_CASE(PROBE_FFMA_LOP3)
        PLIC_PROBE_CASE(PROBE_FFMA2_LOP3)
        PLIC_PROBE_CASE(PROBE_MUFU_FFMA4)
        PLIC_PROBE_CASE(PROBE_FFMA_FMNMX)
        PLIC_PROBE_CASE(PROBE_FSEL)
        PLIC_PROBE_CASE(PROBE_FADD)
        PLIC_PROBE_CASE(PROBE_FMUL)
        PLIC_PROBE_CASE(PROBE_FADD2)
        PLIC_PROBE_CASE(PROBE_3FP_LOP3)
        case plic::PROBE_DFMA:
            plic::pipe_probe_dfma<<<grid, plic::kBlock, 0, stream>>>(sink, trips);
            per_trip = (int64_t)plic::kProbeChains * plic::kProbeUnroll;
            break;
        case plic::PROBE_NESTED_SCALAR:
            plic::pipe_probe_nested_alt<0><<<grid, plic::kBlock, 0, stream>>>(sink, trips);
            per_trip = 4 * 16 * 8;                               // 4 pairs x 16 halvings x 8 instructions
            break;
        case plic::PROBE_NESTED_HYBRID:
            plic::pipe_probe_nested_alt<1><<<grid, plic::kBlock, 0, stream>>>(sink, trips);
            per_trip = 4 * 16 * 6;
            break;
        default:
            plic::pipe_probe_nested<<<grid, plic::kBlock, 0, stream>>>(sink, trips);
            per_trip = 4 * 16 * 5;                               // 4 pairs x 16 halvings x 5 instructions
    }
#undef PLIC_PROBE_CASE
    *warp_instructions = warps * per_trip * trips;
    plic::g_launches.fetch_add(1, std::memory_order_relaxed);
    return cudaPeekAtLastError() == cudaSuccess ? PLIC_OK : PLIC_ERR_LAUNCH;
}

int plic_launch_config(int method, int64_t N, int *grid, int *block, int *cells_per_thread) {
    const int k = method == -1 ? plic::kVolumeKernel : plic::kernel_index(method);
    if (k < 0) return PLIC_ERR_METHOD;
    if (N < 0) return PLIC_ERR_SIZE;
    if (!grid || !block || !cells_per_thread) return PLIC_ERR_NULL;
    cudaError_t err;
    const plic::DeviceInfo *info = plic::device_info(&err);
    if (!info) return PLIC_ERR_LAUNCH;
    *grid = plic::grid_for(N / 4, plic::vec_kernel(k).tiles);
    *block = plic::kBlock;
    *cells_per_thread = 4;
    return PLIC_OK;
}

int64_t plic_launch_count(void) { return plic::g_launches.load(std::memory_order_relaxed); }

}  // extern "C"

#include "plic_curvature_static.cuh"   // plic_curvature_static: the curvature call with a built-in interface list
