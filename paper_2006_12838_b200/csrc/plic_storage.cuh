// plic_storage.cuh -- plic_solve with other storage / arithmetic types:
//
//   binary16 storage, fp32 arithmetic (plic_solve_h, plic_volume_h): 10 B per cell instead of 20.
//       The HBM roofline doubles, so the branch-free packed kernels, which at 20 B per cell leave
//       45 % of the issue slots idle, become bound by instruction issue: this is where the
//       two-cells-per-instruction design is measured against its own ceiling.
//         map_h8           the PLIC_FAST methods, plic_volume_h, blank, kawano: 8 cells per thread,
//                          one 128-bit load per array, conversions binary16 <-> fp32 at the ends;
//         map_compact_io   the four precise methods, as map_compact (plic_kernels.cu): 4 cells
//                          per thread (64-bit loads), heavy cases compacted per tile.
//   fp64 storage and arithmetic (plic_solve_f64): 40 B per cell, the four precise methods of
//       plic_f64.cuh on map_compact_io with 2 cells per thread (128-bit loads).
//
// Included by plic_kernels.cu after the fp32 kernels (uses kBlock, the ld/st helpers, SolveOp,
// VolumeOp, BlankOp, grid_dependency_wait, g_launches).
#pragma once
#include <cuda_fp16.h>

#include "plic_f64.cuh"

namespace plic {

// ---- 128- and 64-bit streaming accesses on raw words ----------------------------------------------
__device__ __forceinline__ uint4 ld_stream_u4(const uint4 *p) {
    uint4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "l"(p));
    return v;
}
__device__ __forceinline__ uint4 ld_stream_rw_u4(const uint4 *p) {       // may alias the output
    uint4 v;
    asm volatile("ld.global.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "l"(p)
                 : "memory");
    return v;
}
// a load ptxas may not drop although its result is unused: the blank run (d0 = V0 - 1/2) ignores the
// normal, but as the ceiling of the access pattern it has to read all four arrays
__device__ __forceinline__ uint4 ld_volatile_u4(const uint4 *p) {
    uint4 v;
    asm volatile("ld.volatile.global.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "l"(p)
                 : "memory");
    return v;
}
template <class OP> struct ReadsNormal { static constexpr bool value = true; };
template <> struct ReadsNormal<BlankOp> { static constexpr bool value = false; };
__device__ __forceinline__ void st_stream_u4(uint4 *p, const uint4 &v) {
    asm volatile("st.global.cs.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w)
                 : "memory");
}
__device__ __forceinline__ uint2 ld_stream_u2(const uint2 *p) {
    uint2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ uint2 ld_stream_rw_u2(const uint2 *p) {
    uint2 v;
    asm volatile("ld.global.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_stream_u2(uint2 *p, const uint2 &v) {
    asm volatile("st.global.cs.v2.u32 [%0], {%1,%2};" ::"l"(p), "r"(v.x), "r"(v.y) : "memory");
}
__device__ __forceinline__ double2 ld_stream_d2(const double2 *p) {
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ double2 ld_stream_rw_d2(const double2 *p) {
    double2 v;
    asm volatile("ld.global.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_stream_d2(double2 *p, const double2 &v) {
    asm volatile("st.global.cs.v2.f64 [%0], {%1,%2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}

// two binary16 values in one 32-bit word <-> two fp32 values (exact / round to nearest even)
__device__ __forceinline__ F2 h2_to_f2(unsigned w) {
    const float2 f = __half22float2(*reinterpret_cast<const __half2 *>(&w));
    return F2{f.x, f.y};
}
__device__ __forceinline__ unsigned f2_to_h2(float lo, float hi) {
    const __half2 h = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<const unsigned *>(&h);
}

// common signature of the body kernels below: n16 = number of 16-byte vectors per array;
// aux: optional fp32 copy of the result before it is rounded to binary16 (binary16 kernels only)
typedef void (*io_kernel_t)(const void *, const void *, const void *, const void *, void *, float *, int64_t);

// ---- map_h8: binary16 storage, packed fp32 arithmetic, 8 cells per thread ---------------------------
// One block per tile of kBlock vectors (2048 cells), handed out by the hardware block scheduler like
// map_vec4.  `s` may be the output array (in-place call).
template <class OP>
__global__ void __launch_bounds__(kBlock, 4)
map_h8(const void *s_, const void *nx_, const void *ny_, const void *nz_, void *out_, float *aux, int64_t n16) {
    grid_dependency_wait();
    const int64_t i = (int64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i >= n16) return;
    const uint4 v = ld_stream_rw_u4(reinterpret_cast<const uint4 *>(s_) + i);
    constexpr bool used = ReadsNormal<OP>::value;
    const uint4 a = used ? ld_stream_u4(reinterpret_cast<const uint4 *>(nx_) + i) : ld_volatile_u4(reinterpret_cast<const uint4 *>(nx_) + i);
    const uint4 b = used ? ld_stream_u4(reinterpret_cast<const uint4 *>(ny_) + i) : ld_volatile_u4(reinterpret_cast<const uint4 *>(ny_) + i);
    const uint4 c = used ? ld_stream_u4(reinterpret_cast<const uint4 *>(nz_) + i) : ld_volatile_u4(reinterpret_cast<const uint4 *>(nz_) + i);
    const unsigned vw[4] = {v.x, v.y, v.z, v.w}, aw[4] = {a.x, a.y, a.z, a.w};
    const unsigned bw[4] = {b.x, b.y, b.z, b.w}, cw[4] = {c.x, c.y, c.z, c.w};
    unsigned rw[4];
    float4 r32[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const F2 v0 = h2_to_f2(vw[2 * h]), v1 = h2_to_f2(vw[2 * h + 1]);
        const F2 a0 = h2_to_f2(aw[2 * h]), a1 = h2_to_f2(aw[2 * h + 1]);
        const F2 b0 = h2_to_f2(bw[2 * h]), b1 = h2_to_f2(bw[2 * h + 1]);
        const F2 c0 = h2_to_f2(cw[2 * h]), c1 = h2_to_f2(cw[2 * h + 1]);
        const float4 r = OP::apply4(make_float4(v0.x, v0.y, v1.x, v1.y), make_float4(a0.x, a0.y, a1.x, a1.y),
                                    make_float4(b0.x, b0.y, b1.x, b1.y), make_float4(c0.x, c0.y, c1.x, c1.y));
        rw[2 * h] = f2_to_h2(r.x, r.y);
        rw[2 * h + 1] = f2_to_h2(r.z, r.w);
        r32[h] = r;
    }
    st_stream_u4(reinterpret_cast<uint4 *>(out_) + i, make_uint4(rw[0], rw[1], rw[2], rw[3]));
    if (aux) {
        st_stream(reinterpret_cast<float4 *>(aux) + 2 * i, r32[0]);
        st_stream(reinterpret_cast<float4 *>(aux) + 2 * i + 1, r32[1]);
    }
}

// ---- arithmetic / storage policies of map_compact_io and map_scalar_io ------------------------------
struct IoF16 {                                   // binary16 in HBM, fp32 in registers
    typedef float real;
    typedef unsigned short elem;
    typedef float4 real4;
    static constexpr int kPer = 4;               // cells per thread: one 64-bit access per array
    static constexpr int kPer16 = 2;             // such accesses per 16-byte vector
    static constexpr int kMinBlocks = 5;
    template <int METHOD> struct Method : Precise<METHOD> {};
    static __device__ __forceinline__ void load(const void *p, int64_t i, bool rw, real (&v)[kPer]) {
        const uint2 *q = reinterpret_cast<const uint2 *>(p) + i;
        const uint2 w = rw ? ld_stream_rw_u2(q) : ld_stream_u2(q);
        const F2 lo = h2_to_f2(w.x), hi = h2_to_f2(w.y);
        v[0] = lo.x; v[1] = lo.y; v[2] = hi.x; v[3] = hi.y;
    }
    static __device__ __forceinline__ void store(void *p, float *aux, int64_t i, const real (&v)[kPer]) {
        st_stream_u2(reinterpret_cast<uint2 *>(p) + i, make_uint2(f2_to_h2(v[0], v[1]), f2_to_h2(v[2], v[3])));
        if (aux) st_stream(reinterpret_cast<float4 *>(aux) + i, make_float4(v[0], v[1], v[2], v[3]));
    }
    static __device__ __forceinline__ real load1(const void *p, int64_t i) {
        return __half2float(__ushort_as_half(reinterpret_cast<const unsigned short *>(p)[i]));
    }
    static __device__ __forceinline__ void store1(void *p, float *aux, int64_t i, real v) {
        reinterpret_cast<unsigned short *>(p)[i] = __half_as_ushort(__float2half_rn(v));
        if (aux) aux[i] = v;
    }
    static __device__ __forceinline__ real4 pack(real a, real b, real c, real d) { return make_float4(a, b, c, d); }
    struct Cell { real n1, n2, n3, V, hS; };
    static __device__ __forceinline__ Cell reduce(real V0, real x, real y, real z) {
        const Reduced r = reduce_cell(V0, x, y, z);
        return Cell{r.n1, r.n2, r.n3, r.V, half_l1(r)};
    }
    static __device__ __forceinline__ real restore(real V0, real hS, real d) { return restore_cell<true>(V0, hS, d); }
};

struct IoF64 {                                   // fp64 in HBM and in registers
    typedef double real;
    typedef double elem;
    typedef double4 real4;
    static constexpr int kPer = 2;               // one 128-bit access per array
    static constexpr int kPer16 = 1;
    static constexpr int kMinBlocks = 4;
    template <int METHOD> struct Method : f64::Precise<METHOD> {};
    static __device__ __forceinline__ void load(const void *p, int64_t i, bool rw, real (&v)[kPer]) {
        const double2 *q = reinterpret_cast<const double2 *>(p) + i;
        const double2 w = rw ? ld_stream_rw_d2(q) : ld_stream_d2(q);
        v[0] = w.x; v[1] = w.y;
    }
    static __device__ __forceinline__ void store(void *p, float *, int64_t i, const real (&v)[kPer]) {
        st_stream_d2(reinterpret_cast<double2 *>(p) + i, make_double2(v[0], v[1]));
    }
    static __device__ __forceinline__ real load1(const void *p, int64_t i) { return reinterpret_cast<const double *>(p)[i]; }
    static __device__ __forceinline__ void store1(void *p, float *, int64_t i, real v) { reinterpret_cast<double *>(p)[i] = v; }
    static __device__ __forceinline__ real4 pack(real a, real b, real c, real d) { return make_double4(a, b, c, d); }
    struct Cell { real n1, n2, n3, V, hS; };
    static __device__ __forceinline__ Cell reduce(real V0, real x, real y, real z) {
        const f64::Reduced r = f64::reduce_cell(V0, x, y, z);
        return Cell{r.n1, r.n2, r.n3, r.V, f64::half_l1(r)};
    }
    static __device__ __forceinline__ real restore(real V0, real hS, real d) { return f64::restore_cell(V0, hS, d); }
};

// ---- map_compact_io: map_compact (plic_kernels.cu) for another storage / arithmetic type -----------
// Same three phases: cheap part for every cell and queueing of the heavy cells, heavy cases (3)/(4)
// and (1) evaluated by dense warps, sign restore and store.  A tile is kPer * kBlock cells.
template <class IO, int METHOD>
__global__ void __launch_bounds__(kBlock, IO::kMinBlocks)
map_compact_io(const void *s, const void *nx, const void *ny, const void *nz, void *out, float *aux, int64_t n16) {
    typedef typename IO::real real;
    typedef typename IO::template Method<METHOD> M;
    constexpr int P = IO::kPer;
    constexpr int kCells = P * kBlock;
    __shared__ typename IO::real4 cells[kCells];     // (n1, n2, n3, V)
    __shared__ real dres[kCells];                    // reduced offset d
    __shared__ unsigned short queue[kCells];
    __shared__ unsigned count;                       // heavy-A entries | heavy-B entries << 16
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    if (tid == 0) count = 0;
    __syncthreads();
    grid_dependency_wait();
    const int64_t nvec = n16 * IO::kPer16;
    const int64_t i = (int64_t)blockIdx.x * kBlock + tid;
    const bool live = i < nvec;
    real V0[P], X[P], Y[P], Z[P];
#pragma unroll
    for (int k = 0; k < P; ++k) {                    // past the end: n = (0, 0, 1), V0 = 0 is case (5) in every
        V0[k] = X[k] = Y[k] = (real)0;               // method, nothing queued (the zero normal would make SZ's
        Z[k] = (real)1;                              // 1/S a NaN and queue the dead slots as heavy cells)
    }
    if (live) {
        IO::load(s, i, true, V0);
        IO::load(nx, i, false, X);
        IO::load(ny, i, false, Y);
        IO::load(nz, i, false, Z);
    }
    real hS[P];
    int kind[P];
    unsigned mine = 0;
#pragma unroll
    for (int k = 0; k < P; ++k) {
        const typename IO::Cell cell = IO::reduce(V0[k], X[k], Y[k], Z[k]);
        hS[k] = cell.hS;
        dres[P * tid + k] = M::cheap(cell.n1, cell.n2, cell.n3, cell.V, kind[k]);
        mine += (unsigned)kind[k];
        cells[P * tid + k] = IO::pack(cell.n1, cell.n2, cell.n3, cell.V);
    }
    unsigned scan = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1)
        asm("{ .reg .pred p; .reg .u32 t; shfl.sync.up.b32 t|p, %0, %1, 0, 0xffffffff; @p add.u32 %0, %0, t; }"
            : "+r"(scan)
            : "r"(o));
    unsigned pos = 0;
    if (lane == 31) pos = atomicAdd(&count, scan);
    pos = __shfl_sync(0xffffffffu, pos, 31) + scan - mine;
#pragma unroll
    for (int k = 0; k < P; ++k) {
        const unsigned idx = kind[k] == KIND_HEAVY_A ? (pos & 0xffffu) : (unsigned)(kCells - 1) - (pos >> 16);
        if (kind[k] != KIND_DONE) queue[idx] = (unsigned short)(P * tid + k);
        pos += (unsigned)kind[k];
    }
    __syncthreads();
    const unsigned na = count & 0xffffu, nb = count >> 16;
    const unsigned na32 = (na + 31u) & ~31u;
    for (unsigned j = tid; j < na32 + nb; j += kBlock) {
        if (j < na32) {
            if (j < na) {
                const unsigned slot = queue[j];
                const typename IO::real4 e = cells[slot];
                dres[slot] = M::heavy_a(e.x, e.y, e.z, e.w);
            }
        } else {
            const unsigned slot = queue[(unsigned)(kCells - 1) - (j - na32)];
            const typename IO::real4 e = cells[slot];
            dres[slot] = M::heavy_b(e.x, e.y, e.z, e.w);
        }
    }
    __syncthreads();
    if (!live) return;
    real r[P];
#pragma unroll
    for (int k = 0; k < P; ++k) r[k] = IO::restore(V0[k], hS[k], dres[P * tid + k]);
    IO::store(out, aux, i, r);
}

// ---- scalar head / tail / misaligned kernels ------------------------------------------------------
template <class OP>                                                  // binary16, any fp32 op of plic_kernels.cu
__global__ void __launch_bounds__(kBlock)
map_scalar_h(const void *s, const void *nx, const void *ny, const void *nz, void *out, float *aux,
             int64_t head, int64_t tail0, int64_t N) {
    const int64_t stride = (int64_t)gridDim.x * kBlock;
    const int64_t count = head + (N - tail0);
    for (int64_t j = (int64_t)blockIdx.x * kBlock + threadIdx.x; j < count; j += stride) {
        const int64_t i = j < head ? j : tail0 + (j - head);
        IoF16::store1(out, aux, i, OP::apply(IoF16::load1(s, i), IoF16::load1(nx, i), IoF16::load1(ny, i), IoF16::load1(nz, i)));
    }
}
template <int METHOD>
__global__ void __launch_bounds__(kBlock)
map_scalar_d(const void *s, const void *nx, const void *ny, const void *nz, void *out, float *,
             int64_t head, int64_t tail0, int64_t N) {
    const int64_t stride = (int64_t)gridDim.x * kBlock;
    const int64_t count = head + (N - tail0);
    for (int64_t j = (int64_t)blockIdx.x * kBlock + threadIdx.x; j < count; j += stride) {
        const int64_t i = j < head ? j : tail0 + (j - head);
        IoF64::store1(out, nullptr, i, f64::solve_cell<METHOD>(IoF64::load1(s, i), IoF64::load1(nx, i), IoF64::load1(ny, i), IoF64::load1(nz, i)));
    }
}
typedef void (*io_scalar_kernel_t)(const void *, const void *, const void *, const void *, void *, float *,
                                   int64_t, int64_t, int64_t);

struct IoBody {
    io_kernel_t fn;          // nullptr: the method has no kernel for this type
    int groups16;            // thread-level accesses per 16-byte vector (grid = ceil(n16 * groups16 / kBlock))
    io_scalar_kernel_t scalar;
};

// k as kernel_index() / kVolumeKernel in plic_kernels.cu
static IoBody io_kernel_h(int k) {
    switch (k) {
        case 0: return IoBody{map_compact_io<IoF16, ANALYTIC>, 2, map_scalar_h<SolveOp<ANALYTIC, false>>};
        case 1: return IoBody{map_compact_io<IoF16, SZ>, 2, map_scalar_h<SolveOp<SZ, false>>};
        case 2: return IoBody{map_compact_io<IoF16, NEWTON>, 2, map_scalar_h<SolveOp<NEWTON, false>>};
        case 3: return IoBody{map_compact_io<IoF16, NESTED>, 2, map_scalar_h<SolveOp<NESTED, false>>};
        case 4: return IoBody{map_h8<SolveOp<ANALYTIC, true>>, 1, map_scalar_h<SolveOp<ANALYTIC, true>>};
        case 5: return IoBody{map_h8<SolveOp<SZ, true>>, 1, map_scalar_h<SolveOp<SZ, true>>};
        case 6: return IoBody{map_h8<SolveOp<NEWTON, true>>, 1, map_scalar_h<SolveOp<NEWTON, true>>};
        case 7: return IoBody{map_h8<SolveOp<NESTED, true>>, 1, map_scalar_h<SolveOp<NESTED, true>>};
        case 8: return IoBody{map_h8<VolumeOp>, 1, map_scalar_h<VolumeOp>};
        case 9: return IoBody{map_h8<SolveOp<KAWANO, false>>, 1, map_scalar_h<SolveOp<KAWANO, false>>};
        case 10: return IoBody{map_h8<BlankOp>, 1, map_scalar_h<BlankOp>};
        default: return IoBody{nullptr, 0, nullptr};
    }
}
static IoBody io_kernel_d(int k) {
    switch (k) {
        case 0: return IoBody{map_compact_io<IoF64, ANALYTIC>, 1, map_scalar_d<ANALYTIC>};
        case 1: return IoBody{map_compact_io<IoF64, SZ>, 1, map_scalar_d<SZ>};
        case 2: return IoBody{map_compact_io<IoF64, NEWTON>, 1, map_scalar_d<NEWTON>};
        case 3: return IoBody{map_compact_io<IoF64, NESTED>, 1, map_scalar_d<NESTED>};
        default: return IoBody{nullptr, 0, nullptr};
    }
}

// elem_bytes = 2 (binary16) or 8 (fp64); aux: optional fp32 copy (binary16 only), 4-byte aligned and,
// for the vector body, congruent to the other pointers in units of cells
static int launch_map_io(const IoBody &body, int elem_bytes, const void *s, const void *nx, const void *ny,
                         const void *nz, void *out, float *aux, int64_t N, cudaStream_t stream) {
    if (N < 0) return PLIC_ERR_SIZE;
    if (!body.fn) return PLIC_ERR_METHOD;
    if (N == 0) return PLIC_OK;
    if (!s || !nx || !ny || !nz || !out) return PLIC_ERR_NULL;
    const uintptr_t ps[5] = {(uintptr_t)s, (uintptr_t)nx, (uintptr_t)ny, (uintptr_t)nz, (uintptr_t)out};
    bool same = true;
    for (int i = 0; i < 5; ++i) {
        if (ps[i] & (uintptr_t)(elem_bytes - 1)) return PLIC_ERR_ALIGN;
        if ((ps[i] & 15u) != (ps[0] & 15u)) same = false;
    }
    if ((uintptr_t)aux & 3u) return PLIC_ERR_ALIGN;
    const int per16 = 16 / elem_bytes;                                   // cells per 16-byte vector
    int64_t head = same ? (int64_t)(((16u - (ps[0] & 15u)) & 15u) / (unsigned)elem_bytes) : N;
    // the fp32 copy is written with 128-bit stores at aux + head: it must be 16-byte aligned there
    if (aux && (((uintptr_t)(aux + head)) & 15u)) head = N;
    if (head > N) head = N;
    const int64_t n16 = (N - head) / per16;
    const int64_t tail0 = head + n16 * per16;
    const char *cs = (const char *)s, *cx = (const char *)nx, *cy = (const char *)ny, *cz = (const char *)nz;
    if (n16 > 0) {
        const int64_t blocks = (n16 * body.groups16 + kBlock - 1) / kBlock;
        if (blocks > 0x7fffffffLL) return PLIC_ERR_SIZE;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)blocks);
        cfg.blockDim = dim3(kBlock);
        cfg.dynamicSmemBytes = 0;
        cfg.stream = stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        const int64_t off = head * elem_bytes;
        if (cudaLaunchKernelEx(&cfg, body.fn, (const void *)(cs + off), (const void *)(cx + off),
                               (const void *)(cy + off), (const void *)(cz + off), (void *)((char *)out + off),
                               aux ? aux + head : (float *)nullptr, n16) != cudaSuccess)
            return PLIC_ERR_LAUNCH;
        g_launches.fetch_add(1, std::memory_order_relaxed);
    }
    const int64_t rest = head + (N - tail0);
    if (rest > 0) {
        const int64_t need = (rest + kBlock - 1) / kBlock;
        body.scalar<<<(int)(need < 0x7fffffffLL ? need : 0x7fffffffLL), kBlock, 0, stream>>>(s, nx, ny, nz, out, aux,
                                                                                         head, tail0, N);
        g_launches.fetch_add(1, std::memory_order_relaxed);
    }
    return cudaPeekAtLastError() == cudaSuccess ? PLIC_OK : PLIC_ERR_LAUNCH;
}

}  // namespace plic
