// plic_curvature.cuh -- curvature from a 3^3 neighbourhood of fill levels (sect. 4, appendix B of
// PAPER.md = /root/reference/PAPER.md): phi_0..phi_26 -> kappa, eq. (41).
//
// Per interface lattice point (0 < phi_0 < 1), in the paper's order:
//   1. Parker-Youngs normal n, eq. (54)/(55)
//   2. basis b_z = n, b_y = (b_z x r)/|.|, b_x = b_y x b_z, eq. (42)-(45)
//   3. for every interface neighbour i: p_i = (e_i.b_x, e_i.b_y, e_i.b_z + d0(phi_i,n) - d0(phi_0,n)),
//      eq. (46) -- this is where PLIC is solved, up to 27 times per point with ONE normal, so the
//      sort, the thresholds and everything else that depends on n alone is computed once
//   4. M = sum Q_i Q_i^T, b = sum z_i Q_i, Q = (x^2, y^2, xy, x, y), eq. (47)-(49), (69)
//   5. M x = b, eq. (70); fewer than 5 points: the leading k x k block
//   6. kappa = (A (I^2+1) + B (H^2+1) - C H I) / (H^2+I^2+1)^(3/2), eq. (63)
//
// Two kernels, because interface points are a 2-D surface in a 3-D lattice (0.4 % of the cells of
// a 256^3 box holding an R = 60 drop):
//   curv_mark4  streams the lattice once (HBM bound: 4 B read + 4 B written per cell), writes
//               kappa = 0 everywhere and appends the index of every interior interface point to a
//               list (one atomicAdd per warp); curv_mark is its scalar form for misaligned lattices;
//   curv_cells  one thread per list entry, so warps are dense: gathers the 27 fill levels (L2
//               hits, the lattice has just been streamed), and runs steps 1-6 in registers; the 26
//               neighbour solves go through the packed two-cells-per-instruction analytic solver.
// Readings C1-C5 of oracle/curvature.py's header apply (sign of kappa, zero for non-interface /
// border / gradient-free / neighbour-free points, reduced rank keeps the first k parameters).
#pragma once
#include "plic_packed.cuh"

namespace plic {

constexpr int kCurvBlock = 64;                 // threads per block of curv_cells

__device__ __forceinline__ bool curv_interior(int64_t i, int nx, int ny, int nz) {
    const unsigned u = (unsigned)i;                               // ncells < 2^31: 32-bit divisions
    const unsigned t = u / (unsigned)nx;
    const int x = (int)(u - t * (unsigned)nx);
    const int z = (int)(t / (unsigned)ny);
    const int y = (int)(t - (unsigned)z * (unsigned)ny);
    return x > 0 && x < nx - 1 && y > 0 && y < ny - 1 && z > 0 && z < nz - 1;
}

// ---- curv_mark -----------------------------------------------------------------------------
// list[0] counts every interior interface point found (also beyond capacity); entries
// list[1 .. min(count, capacity)] hold linear cell indices x + nx (y + ny z).
__global__ void __launch_bounds__(256)
curv_mark(const float *__restrict__ phi, float *__restrict__ kappa, int nx, int ny, int nz,
          int *__restrict__ list, int capacity) {
    const int64_t ncells = (int64_t)nx * ny * nz;
    const int64_t stride = (int64_t)gridDim.x * 256;
    const int lane = threadIdx.x & 31;
    for (int64_t base = (int64_t)blockIdx.x * 256; base < ncells; base += stride) {
        const int64_t i = base + threadIdx.x;
        bool hit = false;
        if (i < ncells) {
            const float p = __ldg(phi + i);
            kappa[i] = 0.0f;
            hit = p > 0.0f && p < 1.0f && curv_interior(i, nx, ny, nz);
        }
        const unsigned m = __ballot_sync(0xffffffffu, hit);
        if (m) {
            int start = 0;
            if (lane == 0) start = atomicAdd(list, __popc(m));
            start = __shfl_sync(0xffffffffu, start, 0);
            const int slot = start + __popc(m & ((1u << lane) - 1u));
            if (hit && slot < capacity) list[1 + slot] = (int)i;
        }
    }
}

// Vector form for 16-byte aligned lattices: four cells per float4 group and kMarkGroups groups in
// flight per thread (64 B loaded before anything is consumed); the ncells % 4 trailing cells are taken
// by the first threads of block 0.  Same list semantics as curv_mark.
// Hits are collected per block in shared memory (warp-aggregated shared atomics) and flushed to the
// global list with one global atomicAdd per block, so that no warp waits for a global atomic's
// round trip inside the streaming loop.  A block that overflows its kMarkCap shared slots appends
// the excess directly to the global list.
constexpr int kMarkCap = 2048;

struct MarkShared {
    int count;
    int base;
    int cells[kMarkCap];
};

__device__ __forceinline__ void curv_append(unsigned hits, int64_t first, MarkShared &sh,
                                            int *__restrict__ list, int capacity) {
    // hits: bit c set = cell first + c is an interior interface point
    const int lane = threadIdx.x & 31;
    const int mine = __popc(hits);
    if (__ballot_sync(0xffffffffu, mine > 0) == 0) return;
    int scan = mine;                                              // inclusive prefix sum over lanes
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, scan, d);
        if (lane >= d) scan += v;
    }
    int start = 0;
    if (lane == 31) start = atomicAdd(&sh.count, scan);
    start = __shfl_sync(0xffffffffu, start, 31);
    int slot = start + scan - mine;
#pragma unroll
    for (int c = 0; c < 4; ++c)
        if (hits & (1u << c)) {
            if (slot < kMarkCap) {
                sh.cells[slot] = (int)(first + c);
            } else {                                              // shared list full: straight to global
                const int g = atomicAdd(list, 1);
                if (g < capacity) list[1 + g] = (int)(first + c);
            }
            ++slot;
        }
}

__device__ __forceinline__ void curv_flush(MarkShared &sh, int *__restrict__ list, int capacity) {
    __syncthreads();
    const int n = sh.count < kMarkCap ? sh.count : kMarkCap;
    if (threadIdx.x == 0 && n > 0) sh.base = atomicAdd(list, n);
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += blockDim.x)
        if (sh.base + i < capacity) list[1 + sh.base + i] = sh.cells[i];
}

constexpr int kMarkGroups = 4;      // float4 groups per thread per step of curv_mark4

__global__ void __launch_bounds__(256)
curv_mark4(const float4 *__restrict__ phi, float4 *__restrict__ kappa, int nx, int ny, int nz,
           int *__restrict__ list, int capacity) {
    const int64_t ncells = (int64_t)nx * ny * nz;
    const int64_t n4 = ncells / 4;
    const int64_t stride = (int64_t)gridDim.x * 256;
    const float4 zero4 = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    __shared__ MarkShared sh;
    if (threadIdx.x == 0) sh.count = 0;
    __syncthreads();
    // whole warps iterate together (the append uses warp collectives): bound by the warp's first lane
    for (int64_t base = (int64_t)blockIdx.x * 256 + (threadIdx.x & ~31); base < n4;
         base += kMarkGroups * stride) {
        int64_t g[kMarkGroups];
        float4 p[kMarkGroups];
#pragma unroll
        for (int k = 0; k < kMarkGroups; ++k) {                      // all loads first
            g[k] = base + (threadIdx.x & 31) + k * stride;
            p[k] = zero4;
            if (g[k] < n4) p[k] = __ldg(phi + g[k]);
        }
#pragma unroll
        for (int k = 0; k < kMarkGroups; ++k)
            if (g[k] < n4) kappa[g[k]] = zero4;
#pragma unroll
        for (int k = 0; k < kMarkGroups; ++k) {
            const float v[4] = {p[k].x, p[k].y, p[k].z, p[k].w};
            unsigned h = 0;
#pragma unroll
            for (int c = 0; c < 4; ++c)
                if (v[c] > 0.0f && v[c] < 1.0f && curv_interior(4 * g[k] + c, nx, ny, nz)) h |= 1u << c;
            curv_append(h, 4 * g[k], sh, list, capacity);
        }
    }
    if (blockIdx.x == 0 && threadIdx.x < 32) {                    // the ncells % 4 trailing cells
        const int64_t i = 4 * n4 + threadIdx.x;
        unsigned h = 0;
        if (i < ncells) {
            const float p = reinterpret_cast<const float *>(phi)[i];
            reinterpret_cast<float *>(kappa)[i] = 0.0f;
            if (p > 0.0f && p < 1.0f && curv_interior(i, nx, ny, nz)) h = 1u;
        }
        curv_append(h, i, sh, list, capacity);
    }
    curv_flush(sh, list, capacity);
}

// ---- steps 1-6 for one point ----------------------------------------------------------------
struct Moments {            // the 12 distinct entries of M (eq. (69)) and the 5 of b
    F2 x4, x2y2, x3y, x3, x2y, y4, xy3, xy2, y3, x2, xy, y2, zx2, zy2, zxy, zx, zy;
};

__device__ __forceinline__ float curvature_point(const float (&p)[27]) {
    // step 1: eq. (54), weights eq. (55); p[(dx+1) + 3 (dy+1) + 9 (dz+1)]
    float g[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) g[a] = 0.0f;
#pragma unroll
    for (int i = 0; i < 27; ++i) {
        const int e[3] = {i % 3 - 1, (i / 3) % 3 - 1, i / 9 - 1};
        const int l1 = (e[0] != 0) + (e[1] != 0) + (e[2] != 0);
        const float w = l1 == 1 ? 4.0f : (l1 == 2 ? 2.0f : 1.0f);
#pragma unroll
        for (int a = 0; a < 3; ++a)
            if (e[a] != 0) g[a] = fmaf(w * (float)e[a], p[i], g[a]);
    }
    const float g2 = fmaf(g[0], g[0], fmaf(g[1], g[1], g[2] * g[2]));
    if (!(g2 > 0.0f)) return 0.0f;                                   // C2
    const float ig = -1.0f / sqrtf(g2);
    const float n[3] = {g[0] * ig, g[1] * ig, g[2] * ig};
    // step 2: eq. (42)-(45)
    const float r[3] = {0.56270900f, 0.32704452f, 0.75921047f};
    float by[3] = {fmaf(n[1], r[2], -n[2] * r[1]), fmaf(n[2], r[0], -n[0] * r[2]),
                   fmaf(n[0], r[1], -n[1] * r[0])};
    const float iby = 1.0f / sqrtf(fmaf(by[0], by[0], fmaf(by[1], by[1], by[2] * by[2])));
    by[0] *= iby; by[1] *= iby; by[2] *= iby;
    const float bx[3] = {fmaf(by[1], n[2], -by[2] * n[1]), fmaf(by[2], n[0], -by[0] * n[2]),
                         fmaf(by[0], n[1], -by[1] * n[0])};
    // step 3: PLIC offsets with the one normal n; the centre's offset first
    const F2 NX{n[0], n[0]}, NY{n[1], n[1]}, NZ{n[2], n[2]};
    const float d00 = solve_pair_fast<ANALYTIC>(F2{p[13], p[13]}, NX, NY, NZ).x;
    Moments s;
    const F2 zero = f2(0.0f);
    s.x4 = s.x2y2 = s.x3y = s.x3 = s.x2y = s.y4 = s.xy3 = s.xy2 = s.y3 = s.x2 = s.xy = s.y2 = zero;
    s.zx2 = s.zy2 = s.zxy = s.zx = s.zy = zero;
    int count = 0;
#pragma unroll
    for (int k = 0; k < 13; ++k) {
        // neighbours in pairs (i0, i1), skipping the centre 13: 0..12 with 14..26 reversed
        const int i0 = k, i1 = 26 - k;
        const F2 ph{p[i0], p[i1]};
        const F2 d0 = solve_pair_fast<ANALYTIC>(ph, NX, NY, NZ);
        const bool u0 = ph.x > 0.0f && ph.x < 1.0f, u1 = ph.y > 0.0f && ph.y < 1.0f;
        count += (int)u0 + (int)u1;
        const F2 m{u0 ? 1.0f : 0.0f, u1 ? 1.0f : 0.0f};
        // e_{i1} = -e_{i0}: the pair sits at opposite ends of one direction
        const int e[3] = {i0 % 3 - 1, (i0 / 3) % 3 - 1, i0 / 9 - 1};
        float px = 0.0f, py = 0.0f, pz = 0.0f;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (e[a] > 0) { px += bx[a]; py += by[a]; pz += n[a]; }
            if (e[a] < 0) { px -= bx[a]; py -= by[a]; pz -= n[a]; }
        }
        const F2 x{px, -px}, y{py, -py};
        const F2 z = add2(F2{pz, -pz}, add2(d0, f2(-d00)));          // eq. (46)
        // step 4: eq. (49), (69); unused points enter with weight m = 0 (their d0 is finite)
        const F2 x2 = mul2(x, x), y2 = mul2(y, y), xy = mul2(x, y);
        const F2 mx2 = mul2(m, x2), my2 = mul2(m, y2), mxy = mul2(m, xy);
        const F2 mx = mul2(m, x), my = mul2(m, y);
        s.x4 = fma2(mx2, x2, s.x4);     s.x2y2 = fma2(mx2, y2, s.x2y2); s.x3y = fma2(mx2, xy, s.x3y);
        s.x3 = fma2(mx2, x, s.x3);      s.x2y = fma2(mx2, y, s.x2y);    s.y4 = fma2(my2, y2, s.y4);
        s.xy3 = fma2(my2, xy, s.xy3);   s.xy2 = fma2(my2, x, s.xy2);    s.y3 = fma2(my2, y, s.y3);
        s.x2 = add2(s.x2, mx2);         s.xy = add2(s.xy, mxy);         s.y2 = add2(s.y2, my2);
        s.zx2 = fma2(mx2, z, s.zx2);    s.zy2 = fma2(my2, z, s.zy2);    s.zxy = fma2(mxy, z, s.zxy);
        s.zx = fma2(mx, z, s.zx);       s.zy = fma2(my, z, s.zy);
    }
    if (count == 0) return 0.0f;                                     // C2
#define PLIC_SUM(f) (s.f.x + s.f.y)
    // symmetric M, eq. (69): only the upper half is formed
    float M[5][5], b[5];
    M[0][0] = PLIC_SUM(x4);  M[0][1] = PLIC_SUM(x2y2); M[0][2] = PLIC_SUM(x3y); M[0][3] = PLIC_SUM(x3);
    M[0][4] = PLIC_SUM(x2y); M[1][1] = PLIC_SUM(y4);   M[1][2] = PLIC_SUM(xy3); M[1][3] = PLIC_SUM(xy2);
    M[1][4] = PLIC_SUM(y3);  M[2][2] = M[0][1];        M[2][3] = M[0][4];       M[2][4] = M[1][3];
    M[3][3] = PLIC_SUM(x2);  M[3][4] = PLIC_SUM(xy);   M[4][4] = PLIC_SUM(y2);
    b[0] = PLIC_SUM(zx2); b[1] = PLIC_SUM(zy2); b[2] = PLIC_SUM(zxy); b[3] = PLIC_SUM(zx); b[4] = PLIC_SUM(zy);
#undef PLIC_SUM
    // fewer than five points: parameters k..4 stay zero -- their rows and columns
    // are replaced by the identity, which leaves the leading k x k block's solution unchanged
#pragma unroll
    for (int i = 1; i < 5; ++i) {
        if (count <= i) {
#pragma unroll
            for (int j = 0; j < 5; ++j)
                if (j < i) M[j][i] = 0.0f; else if (j > i) M[i][j] = 0.0f;
            M[i][i] = 1.0f;
            b[i] = 0.0f;
        }
    }
    // step 5: LU decomposition of the symmetric matrix without pivoting (M is positive definite
    // for points in general position), in the L D L^T form: U = D L^T is kept in the upper half
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const float inv = 1.0f / M[k][k];
#pragma unroll
        for (int i = k + 1; i < 5; ++i) {
            const float f = M[k][i] * inv;                           // L[i][k] (symmetry)
#pragma unroll
            for (int j = i; j < 5; ++j) M[i][j] = fmaf(-f, M[k][j], M[i][j]);
            b[i] = fmaf(-f, b[k], b[i]);
        }
    }
    float xs[5];
#pragma unroll
    for (int i = 4; i >= 0; --i) {
        float acc = b[i];
#pragma unroll
        for (int j = i + 1; j < 5; ++j) acc = fmaf(-M[i][j], xs[j], acc);
        xs[i] = acc / M[i][i];
    }
    // step 6: eq. (63)
    const float A = xs[0], B = xs[1], C = xs[2], H = xs[3], I = xs[4];
    const float w = fmaf(H, H, fmaf(I, I, 1.0f));
    const float num = fmaf(A, fmaf(I, I, 1.0f), fmaf(B, fmaf(H, H, 1.0f), -C * H * I));
    return num / (w * sqrtf(w));
}

// ---- curv_cells ------------------------------------------------------------------------------
__global__ void __launch_bounds__(kCurvBlock)
curv_cells(const float *__restrict__ phi, float *__restrict__ kappa, int nx, int ny,
           const int *__restrict__ list, int capacity) {
    // launched with programmatic stream serialization: the blocks may become resident while
    // curv_mark4 drains; nothing of its output is read before this wait
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int found = list[0];
    const int count = found < capacity ? found : capacity;
    const int64_t sy = nx, sz = (int64_t)nx * ny;
    for (int j = blockIdx.x * kCurvBlock + threadIdx.x; j < count; j += gridDim.x * kCurvBlock) {
        const int64_t c = list[1 + j];
        float p[27];
#pragma unroll
        for (int i = 0; i < 27; ++i)
            p[i] = __ldg(phi + c + (i % 3 - 1) + ((i / 3) % 3 - 1) * sy + (i / 9 - 1) * sz);
        kappa[c] = curvature_point(p);
    }
}

}  // namespace plic
