// plic_curvature_static.cuh -- plic_curvature for callers that cannot provide scratch memory.
//
// plic_curvature needs an interface list (1 + number of interface points int32 values) and leaves
// its allocation to the caller.  Some callers have no way to allocate it:
//   * a flow solver that sized its lattices to fill the GPU at start-up (the VoF-LBM code of
//     PAPER.md sect. 4 is the typical user) has no memory left to ask for when, thousands of time
//     steps later, it wants curvature -- a cudaMalloc there fails, or succeeds today and fails
//     after the next lattice resize;
//   * an application that routes every device allocation through its own pool or accounting layer
//     does not let a library call cudaMalloc behind its back, and may not want to teach its pool
//     about one more buffer just for this;
//   * a time-step loop that must not stall: cudaMalloc and cudaFree synchronise the whole device,
//     so an allocation inside the loop serialises every stream the solver runs.
// For them the list lives in this file, in a device array with static storage duration that is
// part of the library image: the CUDA runtime places it in device memory when the library's
// kernels are loaded onto a GPU and releases it when the process exits.  Nothing is allocated
// by a call; the price is that every GPU the library is used on carries the array (16 MiB) for
// the life of the process, and that the lattice size is limited (PLIC_CURVATURE_STATIC_MAX_POINTS).
//
// Host code cannot use the array's name as a pointer: to the host compiler g_curv_static_list is
// a placeholder object in HOST memory that only identifies the device symbol.  Passing it to a
// kernel hands the GPU a host address (a fault, or on machines whose GPU can reach host memory
// silent use of the wrong bytes).  The device address is a per-device run-time value obtained
// with cudaGetSymbolAddress while that device is current; static_list() below does this once per
// device and keeps the answer.
#pragma once

namespace plic {

constexpr int64_t kStaticEntries = (int64_t)PLIC_CURVATURE_STATIC_MAX_POINTS + 1;   // counter + indices
static_assert(kStaticEntries * sizeof(int) == (size_t)16 << 20, "the static interface list is 16 MiB");

// The interface list of plic_curvature_static: [0] = counter, [1..] = cell indices.  One per GPU,
// shared by every call on that GPU; holds whatever the previous call left in it.
static __device__ __align__(256) int g_curv_static_list[kStaticEntries];

struct StaticList {
    std::mutex mutex;
    int *ptr[kMaxDevices] = {};        // device address of g_curv_static_list on each device, once known
};
static StaticList g_static_list;

// Device address of the list on the CURRENT device, or nullptr if the runtime reports an error.
// The first call per device asks the runtime (which loads the library's device code onto that GPU
// if it is not there yet); later calls return the remembered pointer without touching the runtime
// beyond cudaGetDevice.
static int *static_list() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
        cudaGetLastError();
        return nullptr;
    }
    std::lock_guard<std::mutex> lock(g_static_list.mutex);
    if (g_static_list.ptr[dev]) return g_static_list.ptr[dev];
    int *p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void **)&p, g_curv_static_list);
    if (e != cudaSuccess || !p) {
        cudaGetLastError();            // a failed set-up is retried by the next call
        return nullptr;
    }
    g_static_list.ptr[dev] = p;
    return p;
}

}  // namespace plic

extern "C" int plic_curvature_static(const float *phi, float *kappa, int nx, int ny, int nz,
                                     cudaStream_t stream) {
    // size checks first: they need no device, and a lattice that may not fit is refused before
    // anything is enqueued
    if (nx < 0 || ny < 0 || nz < 0) return PLIC_ERR_SIZE;
    const int64_t ncells = (int64_t)nx * ny * nz;
    if (ncells > 0x7fffffffLL) return PLIC_ERR_SIZE;
    // only cells with a full 3^3 neighbourhood can enter the list
    const int64_t interior = (nx > 2 && ny > 2 && nz > 2) ? (int64_t)(nx - 2) * (ny - 2) * (nz - 2) : 0;
    if (interior > PLIC_CURVATURE_STATIC_MAX_POINTS) return PLIC_ERR_CAPACITY;
    if (ncells > 0 && (!phi || !kappa)) return PLIC_ERR_NULL;
    int *list = plic::static_list();   // also for an empty lattice: such a call is the explicit set-up
    if (!list) return PLIC_ERR_LAUNCH;
    // the caller-scratch path with the static list as its scratch: the same three kernels, the first of
    // which (curv_reset) clears the counter the previous call left behind; stale indices beyond the new
    // count are never read as list entries
    return plic_curvature(phi, kappa, nx, ny, nz, list, plic::kStaticEntries, stream);
}
