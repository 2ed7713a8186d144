/*
 * plic.h -- C ABI of libplic: the batched PLIC plane-cube problem on one B200 (sm_100a).
 *
 * PAPER.md below is /root/reference/PAPER.md, the text of arxiv 2006.12838 ("Analytic
 * Solution to the Piecewise Linear Interface Construction Problem ...").
 *
 * The operation (eq. (1)): for each of N independent cells, a truncated
 * volume V0 in [0,1] and a plane normal n = (nx,ny,nz) are mapped to the plane offset
 *
 *     d0 in [-S/2, +S/2],  S = |nx|+|ny|+|nz|,
 *
 * such that the half-space { x : n.x <= d0 } cuts the volume V0 out of the unit cube
 * [-1/2,1/2]^3 (plic_solve).  plic_volume is the forward map V0(d0, n) of PAPER.md:71-92,
 * eq. (6), (7), (11).  Every step -- mirror/sort (eq. (2)-(4)), volume reduction (eq. (5)),
 * case selection (eq. (26)), the per-case solve (eq. (25), sect. 2.4, 2.5) and the sign
 * restore (eq. (8)) -- runs in hand-written CUDA kernels; there is no CPU fallback.
 *
 * Data layout: structure of arrays, five flat fp32 arrays of N elements each.
 * Algorithmic HBM traffic is 20 B per cell (16 B read, 4 B written).
 */
#ifndef PLIC_H_
#define PLIC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Same opaque type as the CUDA runtime's cudaStream_t (a redeclaration of an identical
 * typedef is legal C11/C++), so this header needs no CUDA include. */
typedef struct CUstream_st *cudaStream_t;

/* ---- method ids: `method` = one of PLIC_METHOD_* optionally OR-ed with PLIC_FAST ---------- */
#define PLIC_METHOD_ANALYTIC 0 /* the paper's analytic inverse: eq. (12), (14)-(26), Listing 2
                                   */
#define PLIC_METHOD_SZ       1 /* Scardovelli-Zaleski solution, edge-case complete and
                                  micro-optimised: sect. 2.4, Listings 3/4 */
#define PLIC_METHOD_NEWTON   2 /* Newton-Raphson for cases (1),(3),(4): sect. 2.5, Listing 6
                                   */
#define PLIC_METHOD_NESTED   3 /* nested intervals (bisection) for cases (3),(4): sect. 2.5,
                                  Listing 5 */
#define PLIC_NUM_METHODS     4 /* the four methods above; each takes PLIC_FAST */
#define PLIC_METHOD_KAWANO   4 /* the SZ solution as translated from Kawano's Fortran, Listing 3
                                  (PAPER.md:187-217), kept for the paper's five-way comparison
                                  and to reproduce its defect: NaN for n = (1,0,0), V0 in {0,1}
                                  (PAPER.md:217, 256).  Not edge-case complete, not accurate for
                                  small normal components; no PLIC_FAST form.  Use PLIC_METHOD_SZ. */
#define PLIC_METHOD_BLANK 0x40 /* the "blank run" of eq. (33): d0 = V0 - 1/2 in place of a PLIC solve
                                  (PAPER.md:241-246).  In plic_roundtrip_error it is the run whose time
                                  the paper subtracts; in plic_solve it is the same 4-read / 1-write
                                  stream with no arithmetic, i.e. the ceiling of the access pattern */
#define PLIC_FAST        0x100 /* approximate SFU roots/reciprocals/trig, branch-free a-priori
                                  case selection, two cells per packed fp32x2 instruction;
                                  without it: IEEE division and square root, CUDA libm
                                  cbrt/asin/acos/sin/cos, cases in the paper's order with the
                                  expensive ones (1), (3), (4) evaluated in dense warps */

/* ---- error codes (functions return 0 on success, never throw, never print) ---------------- */
#define PLIC_OK               0
#define PLIC_ERR_NULL        -1 /* a null pointer with N > 0 */
#define PLIC_ERR_SIZE        -2 /* a size argument is out of range: N < 0, L < 2, work_entries < 2,
                                   negative lattice extents or more than 2^31-1 lattice cells */
#define PLIC_ERR_METHOD      -3 /* unknown method id */
#define PLIC_ERR_LAUNCH      -4 /* the CUDA runtime reported an error (launch, copy, alloc) */
#define PLIC_ERR_ALIGN       -5 /* a pointer is not aligned to its element size (4 bytes for fp32) */
#define PLIC_ERR_CAPACITY    -6 /* plic_curvature_static only: the lattice has more interior cells than
                                   PLIC_CURVATURE_STATIC_MAX_POINTS; nothing was enqueued */

/*
 * plic_solve -- d0[i] = d0(V0[i], n[i]) for i in [0, N)            (eq. (1))
 *
 *   V0, nx, ny, nz  DEVICE pointers, fp32, N elements each, read only.
 *   d0              DEVICE pointer, fp32, N elements, written.  May be the same pointer as
 *                   V0 (each cell is read and then written by the same thread); any other
 *                   overlap is undefined.
 *   N               number of cells, >= 0.  N == 0 is a successful no-op.
 *   method          PLIC_METHOD_* [| PLIC_FAST].
 *   stream          the CUDA stream the work is enqueued on (0 = legacy default stream).
 *
 * The caller owns all memory.  The call allocates nothing, keeps no per-call state, does
 * not synchronise and returns as soon as the kernels are enqueued.  Pointers need only be
 * 4-byte aligned: when all five share one alignment modulo 16 the body runs on 16-byte
 * accesses (bulk asynchronous copies into shared memory or 128-bit loads, 128-bit stores)
 * and at most 3 head + 3 tail cells take a scalar kernel; otherwise the whole range takes
 * the scalar kernel (correct, slower).  Body and scalar kernels give bitwise equal results.
 *
 * Input domain (paper: V0 in [0,1], |n|_2 = 1).  Outside it: V0 < 0 acts as 0, V0 > 1 as 1;
 * n need not be normalised exactly -- every method is written so that
 * d0(V0, c n) = c d0(V0, n) up to rounding; n = (0,0,0) gives d0 = 0.  For every finite
 * input the result is finite (no NaN), including n1 = 0, n1 = n2 = 0 and V0 in {0, 1/2, 1}
 * -- except with PLIC_METHOD_KAWANO, whose NaN at n = (+-1,0,0) (and
 * permutations), V0 in {0, 1} is the point of it.  A NaN input gives an unspecified finite or
 * NaN output.
 *
 * Returns PLIC_OK or a negative PLIC_ERR_*.
 */
int plic_solve(const float *V0, const float *nx, const float *ny, const float *nz,
               float *d0, int64_t N, int method, cudaStream_t stream);

/*
 * plic_volume -- V0[i] = V0(d0[i], n[i]): the forward map ("inverse PLIC", Listing 1,
 * PAPER.md:71-92; eq. (2)-(4), (7), (11), (6)).  Same argument conventions as plic_solve
 * with d0 read and V0 written (V0 may be the same pointer as d0).  |d0| > S/2 (plane misses
 * the cube) gives 0 or 1.  n = (0,0,0) gives 0, 1/2, 1 for d0 <, =, > 0.
 */
int plic_volume(const float *d0, const float *nx, const float *ny, const float *nz,
                float *V0, int64_t N, cudaStream_t stream);

/*
 * plic_solve_h / plic_volume_h -- plic_solve / plic_volume on IEEE binary16 ("half") STORAGE with
 * fp32 ARITHMETIC (the paper itself fixes fp32 storage and arithmetic,
 * PAPER.md:254-256).  10 B of HBM traffic per cell instead of 20, so the HBM roofline doubles and the
 * kernels are bound by instruction issue instead.
 *
 *   V0, nx, ny, nz  DEVICE pointers to N binary16 values each (bit patterns in uint16_t), read only.
 *   d0              DEVICE pointer, N binary16 values, written: the fp32 result of the same arithmetic
 *                   as plic_solve (each input converted exactly), rounded to nearest even.  May be the
 *                   same pointer as V0.
 *   d0_f32          optional DEVICE pointer (NULL to skip), N fp32 values, written: the result BEFORE
 *                   it is rounded to binary16 (+4 B per cell).  d0 is bitwise the rounding of d0_f32.
 *                   This is what the parity tests hold to the 2e-5 bound; d0 itself is within that
 *                   bound plus half a binary16 ulp (2.4e-4 at |d0| in [1/2, 1)).
 *   method          as plic_solve: PLIC_METHOD_* [| PLIC_FAST], PLIC_METHOD_KAWANO, PLIC_METHOD_BLANK.
 *
 * Pointers need only be 2-byte aligned (d0_f32: 4-byte); when the five binary16 pointers share one
 * alignment modulo 16 (and d0_f32 + the head count is 16-byte aligned) the body runs on 128-bit or
 * 64-bit accesses, 8 or 4 cells per thread, otherwise on a scalar kernel with bitwise equal results.
 * Input domain, errors, ownership and stream semantics as plic_solve (PLIC_ERR_ALIGN for an odd
 * address).  The normal as stored is no longer of unit length (binary16 rounding, <= 5e-4 relative);
 * every method is homogeneous in n, so the result is the exact offset for the stored normal.
 */
int plic_solve_h(const uint16_t *V0, const uint16_t *nx, const uint16_t *ny, const uint16_t *nz,
                 uint16_t *d0, float *d0_f32, int64_t N, int method, cudaStream_t stream);
int plic_volume_h(const uint16_t *d0, const uint16_t *nx, const uint16_t *ny, const uint16_t *nz,
                  uint16_t *V0, float *V0_f32, int64_t N, cudaStream_t stream);

/*
 * plic_solve_f64 -- plic_solve in fp64 storage AND arithmetic: 40 B of HBM
 * traffic per cell; IEEE division and square root, CUDA libm cbrt / asin / sin / acos / cos in double
 * precision; the like-for-like GPU counterpart of the fp64 bisection oracle.
 *
 *   V0, nx, ny, nz, d0   DEVICE pointers, fp64, N elements each (d0 may be the same pointer as V0).
 *   method               PLIC_METHOD_ANALYTIC, _SZ, _NEWTON or _NESTED.  There is no PLIC_FAST form
 *                        (the SFU approximations are fp32) and no Kawano / blank method:
 *                        PLIC_ERR_METHOD.
 *
 * Same formulation as the precise fp32 kernels (a-priori case selection, depressed cubics, heavy
 * cases compacted per tile); Newton-Raphson takes 7 steps for cases (3)/(4) and 6 for case (1), nested
 * intervals halves until the fp64 midpoint stops moving.  Pointers must be 8-byte aligned; a common
 * alignment modulo 16 selects the 128-bit body.  Errors, ownership and stream semantics as plic_solve.
 */
int plic_solve_f64(const double *V0, const double *nx, const double *ny, const double *nz, double *d0,
                   int64_t N, int method, cudaStream_t stream);

/*
 * plic_roundtrip_error -- the paper's accuracy and timing benchmark (sect. 2.6):
 * for each of N normals, the volume is varied over [0,1] in L equally spaced steps IN SERIES
 * inside one thread, and
 *
 *     E[i] = (1/L) sum_l | plic_volume(plic_solve(V0_l, n_i), n_i) - V0_l |      (eq. (31))
 *
 * is stored, so that E_avg of eq. (32) is the mean of E over i.  With method =
 * PLIC_METHOD_BLANK the solve is replaced by d0 = V0_l - 1/2 (eq. (33)); the paper's time per
 * PLIC evaluation is (t(method) - t(blank)) / (N L).  The loop reads 12 B and writes 4 B per
 * normal for L evaluations, so unlike plic_solve this entry point is compute bound.
 * The volumes are generated in the kernel: V0_l = fl(l * h) for l = 0..L-2 with
 * h = fl(1 / (L-1)) (fp32 multiplication and division), and V0_{L-1} = 1 exactly
 * (gen.roundtrip_volumes(L) returns the same values).  The sum runs in fp32 over even l and
 * over odd l separately, in increasing l, and the two partial sums are then added.
 *
 *   nx, ny, nz   DEVICE pointers, fp32, N elements each, read only.
 *   E            DEVICE pointer, fp32, N elements, written.
 *   N >= 0, L >= 2;  method = PLIC_METHOD_* [| PLIC_FAST] or PLIC_METHOD_BLANK.
 *
 * Errors, ownership and stream semantics as plic_solve (PLIC_ERR_SIZE also for L < 2).
 */
int plic_roundtrip_error(const float *nx, const float *ny, const float *nz, float *E, int64_t N,
                         int L, int method, cudaStream_t stream);

/*
 * plic_sphere_solve / plic_sphere_volume -- the plane-sphere intersection of sect. 3
 * (PAPER.md:294-321): a sphere of unit volume (radius r = (3/(4 pi))^(1/3), eq. (34)) cut by
 * a plane at offset d0 in [-r, r] from its centre; the direction of the normal is irrelevant.
 *
 *   plic_sphere_volume   V0[i] = pi/3 (r + d0[i])^2 (2r - d0[i])                  (eq. (37))
 *   plic_sphere_solve    d0[i] = the offset with that volume, eq. (38)           (eq. (36))
 *
 * DEVICE pointers, fp32, N elements each; the output may be the same pointer as the input.
 * fast = 0: IEEE sqrt and CUDA libm asin/sin/cos; fast = PLIC_FAST: SFU square roots and the
 * polynomial sin(asin(.)/3) of the cube kernels.  V0 < 0 acts as 0, V0 > 1 as 1; |d0| > r gives
 * 0 or 1.  8 B of HBM traffic per cell.  Errors, alignment, ownership and stream semantics as
 * plic_solve (PLIC_ERR_METHOD for any other value of fast).
 */
int plic_sphere_solve(const float *V0, float *d0, int64_t N, int fast, cudaStream_t stream);
int plic_sphere_volume(const float *d0, float *V0, int64_t N, cudaStream_t stream);

/*
 * plic_curvature -- mean curvature of the interface from fill levels (sect. 4 and appendix B,
 * PAPER.md:323-393, 510-614; eq. (41): phi_0..phi_26 -> kappa).  For every interface lattice point
 * (0 < phi < 1) with a full 3^3 neighbourhood: Parker-Youngs normal (eq. (54), (55)), basis
 * (eq. (42)-(45)), PLIC-corrected neighbour points (eq. (46), analytic PLIC solve with the centre's
 * normal, interface neighbours only), least-squares paraboloid (eq. (47)-(49), (69), (70); with k < 5
 * points only the first k of (A, B, C, H, I) are fitted), kappa by eq. (63).
 *
 *   phi      DEVICE pointer, fp32, nx*ny*nz fill levels, index x + nx (y + ny z), read only.
 *   kappa    DEVICE pointer, fp32, same shape, written: eq. (63) at interface points, 0 at every
 *            other cell (also at interface points on the lattice border, with a vanishing
 *            gradient sum, or without interface neighbours).  Must not overlap phi.
 *   work     DEVICE pointer to work_entries int32 of scratch owned by the caller.  On return
 *            (after the stream has run) work[0] = number of interface points found and
 *            work[1..] their cell indices, in no particular order.  work_entries >= 1 + that
 *            number is required for a complete result (1 + nx*ny*nz always suffices); points
 *            beyond the capacity keep kappa = 0, which the caller can detect from work[0].
 *   nx, ny, nz >= 0, nx*ny*nz < 2^31.
 *
 * Sign: with the normal of eq. (54) pointing out of the fluid, eq. (63) is negative for a convex
 * fluid body (-1/R for a drop of radius R) and positive for a bubble.
 * Rank deficiency: the paper solves eq. (70) by LU decomposition without a pivot check.  Here a fit
 * parameter whose pivot falls below 1e-6 of its diagonal entry of M (the points do not determine it:
 * a lone neighbour, neighbours on one line or coplanar with the normal, coincident abscissae) is
 * dropped like the parameters beyond the number of points: it stays 0 and takes no part
 * in the elimination.  kappa is therefore finite for every finite lattice.
 * Three kernels are enqueued on `stream`, each a programmatic dependent launch of its predecessor: the
 * reset of the list counter, a streaming pass (128-bit accesses when phi and kappa are 16-byte aligned,
 * scalar otherwise) and a dense pass over the interface list, one thread per point.  Aligned and
 * unaligned calls give bitwise the same kappa.  Errors, ownership and stream semantics as plic_solve.
 */
int plic_curvature(const float *phi, float *kappa, int nx, int ny, int nz, int32_t *work,
                   int64_t work_entries, cudaStream_t stream);

/*
 * plic_curvature_static -- plic_curvature without a `work` argument, for callers that cannot allocate
 * device memory at the point where they need curvature.
 *
 * Who that is: a flow solver that gave all of the GPU's memory to its lattices at start-up and has
 * nothing left to ask for (a cudaMalloc deep into a run fails, or starts failing after the next lattice
 * resize); an application whose device memory is managed by its own pool or accounting layer, which a
 * library must not bypass; a time-step loop that cannot afford cudaMalloc / cudaFree, both of which
 * synchronise the whole device and stall every stream.  plic_curvature asks such a caller for scratch
 * it cannot produce.  Here the interface list is a fixed array inside the library instead: it is part
 * of the library's device image, so a GPU holds it (16 MiB) from the moment the library's device code
 * is loaded onto it until the process exits, whether or not this function is ever called again.  The
 * call itself allocates and frees nothing, directly or through any library routine.
 *
 *   phi, kappa, nx, ny, nz, stream   exactly as plic_curvature; the caller still owns input and output.
 *
 * Limit: the list holds PLIC_CURVATURE_STATIC_MAX_POINTS cell indices.  Only cells with a full 3^3
 * neighbourhood are listed, so a lattice is accepted when (nx-2)(ny-2)(nz-2) does not exceed that
 * number -- e.g. up to 163^3, or 1026 x 1026 x 6 -- and the result is then always complete (bitwise the
 * kappa of plic_curvature with a large enough `work`).  A larger lattice is refused with
 * PLIC_ERR_CAPACITY before anything is enqueued, even if it happens to contain few interface cells:
 * use plic_curvature with caller-owned scratch for those.
 *
 * First call on each device: the function looks up the array's device address (cudaGetSymbolAddress,
 * with that device current; the CUDA runtime may load the library's device code onto the GPU at this
 * moment) and remembers it.  Make that first call during start-up, outside any stream capture and
 * before the phase in which allocation is impossible; a call with an empty lattice
 * (nx = 0, phi = kappa = NULL) does the look-up and nothing else.  If the look-up fails the call returns
 * PLIC_ERR_LAUNCH and the next call tries again.
 *
 * One list per GPU, shared by every call: the list still holds the previous call's entries when the
 * next call starts (the call's first kernel clears the counter, which is all that has to start at
 * zero).  Two calls on the same GPU whose kernels can overlap -- different streams without an event
 * between them, or several host threads -- race on the list and give wrong kappa.  Calls on one stream,
 * or ordered by events, are safe; so are calls on different GPUs.  The interface count and list are not
 * returned; a caller that needs them uses plic_curvature.
 *
 * Returns PLIC_OK, PLIC_ERR_SIZE (negative extents, >= 2^31 cells), PLIC_ERR_CAPACITY, PLIC_ERR_NULL,
 * PLIC_ERR_ALIGN or PLIC_ERR_LAUNCH.
 */
#define PLIC_CURVATURE_STATIC_MAX_POINTS 4194303 /* 2^22 - 1: with the counter, 16 MiB of int32 */
int plic_curvature_static(const float *phi, float *kappa, int nx, int ny, int nz, cudaStream_t stream);

/*
 * plic_solve_host / plic_volume_host -- the same maps for HOST arrays (pageable or pinned;
 * pinned memory makes the copies asynchronous).  The range is cut into chunks; host->device
 * copies, the kernel and the device->host copy of consecutive chunks overlap on three
 * internal streams of the current device.  Synchronous: the result is complete in d0 / V0
 * when the call returns.  A device workspace (3 x 5 x chunk fp32) is allocated on first use
 * per device, kept for later calls and freed by plic_host_release().  Not re-entrant: calls
 * from several host threads are serialised by an internal lock.
 */
int plic_solve_host(const float *V0, const float *nx, const float *ny, const float *nz,
                    float *d0, int64_t N, int method);
int plic_volume_host(const float *d0, const float *nx, const float *ny, const float *nz,
                     float *V0, int64_t N);
/* Frees the host-API workspace and streams of every device; safe to call at any time. */
void plic_host_release(void);

/* "analytic", "sz", "newton", "nested" (+ "-fast" with PLIC_FAST), "kawano", "blank"; NULL if
 * unknown.
 * The string is static storage owned by the library. */
const char *plic_method_name(int method);

/* Static text for a PLIC_ERR_* code (never NULL). */
const char *plic_error_string(int code);

/* ABI version: 100*major + minor (1.04: + plic_roundtrip_error, plic_sphere_*, plic_curvature,
 * PLIC_METHOD_KAWANO; 1.05: + plic_solve_h, plic_volume_h, plic_solve_f64, PLIC_METHOD_BLANK in
 * plic_solve; 1.06: + plic_curvature_static, PLIC_ERR_CAPACITY). */
int plic_version(void);

/*
 * plic_pipe_probe -- measurement support for the roofline denominators ("the
 * builder must confirm [the per-SM rates] with an FFMA-only and a MUFU-only microbenchmark").
 * Enqueues one launch of a kernel that executes a single kind of instruction in independent
 * dependency chains (16 warps per SM sub-partition, SM count x 8 blocks of 256 threads) and
 * stores in *warp_instructions (HOST pointer) how many warp-instructions of that kind the launch
 * executes; the caller times the launch (CUDA events) and divides.
 *   pipe  0 scalar FFMA, 1 packed FFMA2, 2 MUFU (rsqrt), 3 FMNMX (ALU pipe), 4 LOP3 (ALU pipe),
 *         5 the halving step of nested-fast (2 FFMA2 + 2 LOP3 + FADD2 per pair), 6-16 mixes of these
 *         (names in the Python binding's PROBES), 17 fp64 FMA
 *   trips loop trips per thread, >= 0 (64 instructions per chain set and trip; 320 for pipe 5)
 *   sink  DEVICE pointer to >= 256 floats (never written in practice; keeps the chains alive)
 * Returns PLIC_OK or PLIC_ERR_METHOD (unknown pipe) / _SIZE / _NULL / _LAUNCH.
 */
int plic_pipe_probe(int pipe, int trips, float *sink, int64_t *warp_instructions, cudaStream_t stream);

/*
 * plic_launch_config -- the launch geometry plic_solve (method >= 0) or plic_volume
 * (method == -1) uses for N cells with 16-byte aligned pointers on the current device:
 * *grid thread blocks of *block threads, each thread handling *cells_per_thread cells of each
 * tile its block owns (one or two tiles per block).  For reporting only.  Returns PLIC_OK or an error code.
 */
int plic_launch_config(int method, int64_t N, int *grid, int *block, int *cells_per_thread);

/* Number of kernels this library has launched in this process since load (all threads). */
int64_t plic_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* PLIC_H_ */
