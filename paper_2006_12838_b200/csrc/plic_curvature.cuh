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
// Interface points are a 2-D surface in a 3-D lattice (0.4 % of the cells of a 256^3 box holding an
// R = 60 drop), so a thread per lattice cell would run the ~2000-instruction point routine in warps
// with one or two active lanes.  Two passes instead (three launches per call, chained as programmatic
// dependent launches; curv_reset clears the list counter first):
//   curv_mark4  streams the lattice once (HBM bound: 4 B read + 4 B written per cell), writes
//               kappa = 0 everywhere and collects the interior interface points per block in shared
//               memory (warp-aggregated), flushed to the caller's list with one global atomicAdd per
//               block; curv_mark is its scalar form for lattices off the 16-byte boundary;
//   curv_cells  the list entries in dense warps, kPointLanes lanes per point (1 by default; 2 and 4 are
//               kept as template instances: the 13 neighbour pairs (e, -e) and the centre are dealt to
//               the lanes of a point, gradient sums and moments reduced with xor shuffles).  A lane
//               gathers its fill levels (L2 hits, the lattice has just been streamed), solves its PLIC
//               offsets with the packed analytic solver and accumulates its share of the 17 moments.
//               Measured on the 256^3 / R = 60 lattice: every split that keeps
//               the registers is equal within 0.2 us -- more lanes shorten one point's dependent chain
//               but add waves -- so the pass is bound by one point's latency, not by throughput.
//               (Evaluating the points inside the streaming kernel -- each block its own -- was tried:
//               49 us per call instead of 38, the point routine's registers cut the streaming
//               occupancy and every block with a single point pays a full round.)
// Readings C1-C5 of oracle/curvature.py's header apply (sign of kappa, zero for non-interface /
// border / gradient-free / neighbour-free points, reduced rank keeps the first k parameters).
#pragma once
#include "plic_packed.cuh"

// ---- tuning switches of the point pass (curvature_point, curv_cells) --------------------------------
// Defined here, ahead of every use: an `#if` on a macro that is only defined further down silently takes
// the 0 branch (this is how round 2 shipped KEEP = 0 while the text said 1).
#ifndef PLIC_CURV_KEEP
#define PLIC_CURV_KEEP 1     // keep the 26 fill levels in registers between step 1 and step 3 (0: read them again, L1 hits)
#endif
#ifndef PLIC_CURV_LANES
#define PLIC_CURV_LANES 1
#endif
#ifndef PLIC_CURV_BLOCK
#define PLIC_CURV_BLOCK 64
#endif
#ifndef PLIC_CURV_MINBLOCKS
#define PLIC_CURV_MINBLOCKS 7
#endif
#if PLIC_CURV_KEEP != 0 && PLIC_CURV_KEEP != 1
#error "PLIC_CURV_KEEP must be 0 or 1"
#endif

namespace plic {


__device__ __forceinline__ bool curv_interior(int64_t i, int nx, int ny, int nz) {
    const unsigned u = (unsigned)i;                               // ncells < 2^31: 32-bit divisions
    const unsigned t = u / (unsigned)nx;
    const int x = (int)(u - t * (unsigned)nx);
    const int z = (int)(t / (unsigned)ny);
    const int y = (int)(t - (unsigned)z * (unsigned)ny);
    return x > 0 && x < nx - 1 && y > 0 && y < ny - 1 && z > 0 && z < nz - 1;
}

// ---- curv_reset ----------------------------------------------------------------------------
// Clears the list counter.  A kernel (not a memset) so that the three launches of a call form one
// chain of programmatic dependent launches: each becomes resident while its predecessor drains and
// touches global memory only after griddepcontrol.wait, i.e. after the predecessor has completed.
__global__ void curv_reset(int *__restrict__ list) {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (threadIdx.x == 0) list[0] = 0;
}

// ---- curv_mark -----------------------------------------------------------------------------
// list[0] counts every interior interface point found (also beyond capacity); entries
// list[1 .. min(count, capacity)] hold linear cell indices x + nx (y + ny z).
__global__ void __launch_bounds__(256)
curv_mark(const float *__restrict__ phi, float *__restrict__ kappa, int nx, int ny, int nz,
          int *__restrict__ list, int capacity) {
    asm volatile("griddepcontrol.wait;" ::: "memory");
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
    asm volatile("griddepcontrol.wait;" ::: "memory");           // before the first global access
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
                if (v[c] > 0.0f && v[c] < 1.0f) h |= 1u << c;
            // interface cells are rare: the interior test (two integer divisions per cell) and the
            // append run only in warps that hold one
            if (__ballot_sync(0xffffffffu, h != 0) == 0) continue;
#pragma unroll
            for (int c = 0; c < 4; ++c)
                if ((h & (1u << c)) && !curv_interior(4 * g[k] + c, nx, ny, nz)) h &= ~(1u << c);
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

// ---- steps 1-6 for one point, on LANES adjacent lanes ---------------------------------------------
// sub = lane % LANES (LANES = 2 or 4).  Slot s of a lane holds item = sub + LANES s: items 0..12 are the
// neighbour pairs (e_k, -e_k), e_k = (k % 3 - 1, (k / 3) % 3 - 1, k / 9 - 1); item 13 is the centre (its
// offset d0(phi_0, n) is broadcast to the group from lane sub = 1); items 14, 15 (LANES = 4) repeat pairs
// with weight 0.  All 32 lanes of the warp must call this together (shuffles); `c` must be an interior
// cell for every lane.
// Symmetry of a pair: x, y flip sign with e, so with the weights m+, m- (1 for an interface neighbour)
// the even moments take (m+ + m-), the odd ones (m+ - m-), and the z-moments m+ z+ +- m- z-.
constexpr float kPivotRel = 1e-6f;     // a pivot below this fraction of its diagonal entry drops the parameter

template <int LANES>
__device__ __forceinline__ float curvature_point(const float *__restrict__ phi, int64_t c, int64_t sy,
                                                 int64_t sz, int sub) {
    static_assert(LANES == 1 || LANES == 2 || LANES == 4, "13 pairs + the centre on 1, 2 or 4 lanes");
    constexpr int SLOTS = (14 + LANES - 1) / LANES;                  // 7 or 4
    const unsigned full = 0xffffffffu;
    const float *pc = phi + c;
    const int isy = (int)sy, isz = (int)sz;                          // ncells < 2^31
    float g[3] = {0.0f, 0.0f, 0.0f};
#if PLIC_CURV_KEEP
    float keep_p[SLOTS], keep_m[SLOTS];
#endif
    // step 1: eq. (54), weights eq. (55): 4, 2, 1 for |e|_1 = 1, 2, 3; the pair contributes w e (phi+ - phi-).
    // PLIC_CURV_KEEP = 1: the 26 fill levels stay in registers for step 3; 0: step 3 reads them again
    // (L1 hits), which frees ~35 registers.
#pragma unroll
    for (int s = 0; s < SLOTS; ++s) {
        const int k = sub + LANES * s;
        const int t = (k * 11) >> 5;                                 // k / 3 for k <= 15
        const int ex = k - 3 * t - 1, ey = t - (t >= 3 ? 3 : 0) - 1, ez = (k >= 9 ? 1 : 0) - 1;
        const int off = ex + ey * isy + ez * isz;
        const int l1 = (ex != 0) + (ey != 0) + (ez != 0);
#if PLIC_CURV_KEEP
        keep_p[s] = __ldg(pc + off);
        keep_m[s] = __ldg(pc - off);
        const float w = k < 13 ? (float)(8 >> l1) * (keep_p[s] - keep_m[s]) : 0.0f;
#else
        const float w = k < 13 ? (float)(8 >> l1) * (__ldg(pc + off) - __ldg(pc - off)) : 0.0f;
#endif
        g[0] = fmaf(w, (float)ex, g[0]);
        g[1] = fmaf(w, (float)ey, g[1]);
        g[2] = fmaf(w, (float)ez, g[2]);
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (LANES >= 2) g[a] += __shfl_xor_sync(full, g[a], 1);
        if (LANES == 4) g[a] += __shfl_xor_sync(full, g[a], 2);
    }
    const float g2 = fmaf(g[0], g[0], fmaf(g[1], g[1], g[2] * g[2]));
    const bool has_normal = g2 > 0.0f;                               // C2 otherwise
    const float ig = has_normal ? -1.0f / sqrtf(g2) : 0.0f;
    const float n[3] = {has_normal ? g[0] * ig : 0.0f, has_normal ? g[1] * ig : 0.0f, has_normal ? g[2] * ig : 1.0f};
    // step 2: eq. (42)-(45)
    const float r[3] = {0.56270900f, 0.32704452f, 0.75921047f};
    float by[3] = {fmaf(n[1], r[2], -n[2] * r[1]), fmaf(n[2], r[0], -n[0] * r[2]),
                   fmaf(n[0], r[1], -n[1] * r[0])};
    const float iby = rsqrtf(fmaxf(fmaf(by[0], by[0], fmaf(by[1], by[1], by[2] * by[2])), 1e-30f));
    by[0] *= iby; by[1] *= iby; by[2] *= iby;
    const float bx[3] = {fmaf(by[1], n[2], -by[2] * n[1]), fmaf(by[2], n[0], -by[0] * n[2]),
                         fmaf(by[0], n[1], -by[1] * n[0])};
    // step 3: PLIC offsets with the one normal n (packed pair = the two ends of one direction)
    const F2 NX{n[0], n[0]}, NY{n[1], n[1]}, NZ{n[2], n[2]};
    float x4 = 0.f, x2y2 = 0.f, x3y = 0.f, x3 = 0.f, x2y = 0.f, y4 = 0.f, xy3 = 0.f, xy2 = 0.f, y3 = 0.f;
    float sx2 = 0.f, sxy = 0.f, sy2 = 0.f, zx2 = 0.f, zy2 = 0.f, zxy = 0.f, zx = 0.f, zy = 0.f;
    int count = 0;
    float d00 = 0.0f;
#pragma unroll
    for (int q = 0; q < SLOTS; ++q) {
        const int s = q == 0 ? SLOTS - 1 : q - 1;                    // the last slot first: it holds the centre
        const int k = sub + LANES * s;
        const int t = (k * 11) >> 5;
        const int ex = k - 3 * t - 1, ey = t - (t >= 3 ? 3 : 0) - 1, ez = (k >= 9 ? 1 : 0) - 1;
        const int off = ex + ey * isy + ez * isz;
#if PLIC_CURV_KEEP
        const float pp = keep_p[s], pm = keep_m[s];
#else
        const float pp = __ldg(pc + off), pm = __ldg(pc - off);
#endif
        const F2 d0 = solve_pair_fast<ANALYTIC>(F2{pp, pm}, NX, NY, NZ);
        if (q == 0) d00 = LANES == 1 ? d0.x : __shfl_sync(full, d0.x, (threadIdx.x & (32 - LANES)) | 1);   // from lane sub = 1
        const bool u0 = k < 13 && pp > 0.0f && pp < 1.0f, u1 = k < 13 && pm > 0.0f && pm < 1.0f;
        count += (int)u0 + (int)u1;
        const float m0 = u0 ? 1.0f : 0.0f, m1 = u1 ? 1.0f : 0.0f;
        const float fx = (float)ex, fy = (float)ey, fz = (float)ez;
        const float px = fmaf(fx, bx[0], fmaf(fy, bx[1], fz * bx[2]));
        const float py = fmaf(fx, by[0], fmaf(fy, by[1], fz * by[2]));
        const float pz = fmaf(fx, n[0], fmaf(fy, n[1], fz * n[2]));
        const float z0 = m0 * (pz + (d0.x - d00)), z1 = m1 * ((d0.y - d00) - pz);      // eq. (46), weighted
        const float ms = m0 + m1, md = m0 - m1, zs = z0 + z1, zd = z0 - z1;
        // step 4: eq. (49), (69)
        const float x2 = px * px, y2 = py * py, xy = px * py;
        const float ex2 = ms * x2, ey2 = ms * y2, exy = ms * xy, ox2 = md * x2, oy2 = md * y2;
        x4 = fmaf(ex2, x2, x4);    x2y2 = fmaf(ex2, y2, x2y2); x3y = fmaf(ex2, xy, x3y);
        y4 = fmaf(ey2, y2, y4);    xy3 = fmaf(ey2, xy, xy3);
        x3 = fmaf(ox2, px, x3);    x2y = fmaf(ox2, py, x2y);   xy2 = fmaf(oy2, px, xy2);  y3 = fmaf(oy2, py, y3);
        sx2 += ex2;                sxy += exy;                 sy2 += ey2;
        zx2 = fmaf(zs, x2, zx2);   zy2 = fmaf(zs, y2, zy2);    zxy = fmaf(zs, xy, zxy);
        zx = fmaf(zd, px, zx);     zy = fmaf(zd, py, zy);
    }
#define PLIC_REDUCE4(v) if (LANES >= 2) v += __shfl_xor_sync(full, v, 1); if (LANES == 4) v += __shfl_xor_sync(full, v, 2);
    PLIC_REDUCE4(x4) PLIC_REDUCE4(x2y2) PLIC_REDUCE4(x3y) PLIC_REDUCE4(x3) PLIC_REDUCE4(x2y) PLIC_REDUCE4(y4)
    PLIC_REDUCE4(xy3) PLIC_REDUCE4(xy2) PLIC_REDUCE4(y3) PLIC_REDUCE4(sx2) PLIC_REDUCE4(sxy) PLIC_REDUCE4(sy2)
    PLIC_REDUCE4(zx2) PLIC_REDUCE4(zy2) PLIC_REDUCE4(zxy) PLIC_REDUCE4(zx) PLIC_REDUCE4(zy) PLIC_REDUCE4(count)
#undef PLIC_REDUCE4
    // symmetric M, eq. (69): only the upper half is formed
    float M[5][5], b[5];
    M[0][0] = x4;  M[0][1] = x2y2; M[0][2] = x3y; M[0][3] = x3;  M[0][4] = x2y;
    M[1][1] = y4;  M[1][2] = xy3;  M[1][3] = xy2; M[1][4] = y3;
    M[2][2] = x2y2; M[2][3] = x2y; M[2][4] = xy2;
    M[3][3] = sx2; M[3][4] = sxy;  M[4][4] = sy2;
    b[0] = zx2; b[1] = zy2; b[2] = zxy; b[3] = zx; b[4] = zy;
    // step 5: LU decomposition of the symmetric positive semi-definite matrix without pivoting, in the
    // L D L^T form (U = D L^T is kept in the upper half).  A parameter is dropped (stays 0, and takes no
    // part in the elimination) when fewer points than its index + 1 were used ("reducing
    // dimensionality"), or when its pivot has fallen below kPivotRel of its diagonal entry -- the
    // points then do not determine it (coplanar with the normal, coincident abscissae); the paper's LU
    // has no such check, the result without it would be Inf or NaN.
    float inv[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const float diag = k == 0 ? x4 : (k == 1 ? y4 : (k == 2 ? x2y2 : (k == 3 ? sx2 : sy2)));
        const bool keep = count > k && M[k][k] > kPivotRel * diag;
        inv[k] = keep ? 1.0f / M[k][k] : 0.0f;
#pragma unroll
        for (int i = k + 1; i < 5; ++i) {
            const float f = M[k][i] * inv[k];                        // L[i][k] (symmetry)
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
        xs[i] = acc * inv[i];
    }
    // step 6: eq. (63)
    const float A = xs[0], B = xs[1], C = xs[2], H = xs[3], I = xs[4];
    const float w = fmaf(H, H, fmaf(I, I, 1.0f));
    const float num = fmaf(A, fmaf(I, I, 1.0f), fmaf(B, fmaf(H, H, 1.0f), -C * H * I));
    const float kap = num / (w * sqrtf(w));
    // C2; a fit whose parameters overflow fp32 (pivots just above the guard) also gives 0, never Inf or NaN
    return (has_normal && count > 0 && fabsf(kap) < 3.0e38f) ? kap : 0.0f;
}

// ---- curv_cells: kPointLanes lanes per entry of the caller's list ------------------------------------
constexpr int kPointLanes = PLIC_CURV_LANES;
constexpr int kCurvBlock = PLIC_CURV_BLOCK;    // threads per block

__global__ void __launch_bounds__(kCurvBlock, PLIC_CURV_MINBLOCKS)
curv_cells(const float *__restrict__ phi, float *__restrict__ kappa, int nx, int ny,
           const int *__restrict__ list, int capacity) {
    // launched with programmatic stream serialization: the blocks may become resident while
    // curv_mark drains; nothing of its output is read before this wait
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int sub = threadIdx.x % kPointLanes;
    const int per = kCurvBlock / kPointLanes;
    // the count and this thread's first list entry are independent loads: one memory round trip, not two
    const int jfirst = blockIdx.x * per + threadIdx.x / kPointLanes;
    const int found = list[0];
    int cfirst = list[1 + (jfirst < capacity ? jfirst : 0)];        // capacity >= 1; stale beyond the count, unused then
    const int count = found < capacity ? found : capacity;
    const int64_t sy = nx, sz = (int64_t)nx * ny;
    for (int j0 = blockIdx.x * per; j0 < count; j0 += gridDim.x * per) {     // uniform per block
        const int j = j0 + threadIdx.x / kPointLanes;
        const bool live = j < count;
        const int64_t c = (j == jfirst && live) ? cfirst : list[1 + (live ? j : count - 1)];
        const float k = curvature_point<kPointLanes>(phi, c, sy, sz, sub);
        if (live && sub == 0) kappa[c] = k;
    }
}

}  // namespace plic
