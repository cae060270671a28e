// noalloc.cu -- gn_nav_compute_step_noalloc: gn_nav_compute_step for callers that must not allocate (code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// gn_nav_compute_step groups the queries of a general geometry by volume key before ComputeStep (SURVEY 8(a) A10 applied to
// A11, common.cuh) and takes the scratch of that sort -- key totals and cursors, one key byte and one work-order index per
// query -- from the handle's stream-ordered memory pool.  Here the same kernels get the same scratch from ONE file-scope
// array in device memory, of a fixed size: every GPU that loads the library holds GN_NOALLOC_SCRATCH_BYTES (5.3 MB) until the
// process exits, and a call is limited to GN_NOALLOC_MAX_QUERIES queries.  No cudaMalloc, cudaFree or pool call is made.
//
// The array's name is a host-side stand-in in host code, not a device address: its device address is looked up once per
// device with cudaGetSymbolAddress (that device current) and kept; the kernels receive that pointer.
// All calls share the array and it keeps the last call's contents: the counters are cleared at the start of every call
// (keys and the work order are fully overwritten before they are read), and two calls that overlap on the GPU (different
// streams, or different host threads on different streams) race on it -- callers serialise them.
#include <mutex>
#include "common.cuh"
#include "nav_kernels.cuh"

namespace gn {

constexpr int64_t NOALLOC_MAX_QUERIES = GN_NOALLOC_MAX_QUERIES;
constexpr size_t NOALLOC_HEAD = STEP_SORT_HEAD;                        // totals and cursors of the two work orders (4 x 32 x u64)
constexpr size_t NOALLOC_BYTES = NOALLOC_HEAD + (size_t)NOALLOC_MAX_QUERIES + 4 * (size_t)NOALLOC_MAX_QUERIES;
static_assert(NOALLOC_BYTES == GN_NOALLOC_SCRATCH_BYTES, "gammanav.h states the size of the scratch array");
static_assert(NOALLOC_HEAD == 1024 && SORT_KEYS2 <= SORT_KEYS_MAX && NOALLOC_MAX_QUERIES % 64 == 0, "scratch layout");

static __device__ __align__(256) unsigned char noalloc_scratch[NOALLOC_BYTES];

// device address of the array on each device, looked up on first use with that device current
constexpr int NOALLOC_MAX_DEVICES = 64;
static std::mutex noalloc_mutex;
static unsigned char* noalloc_ptr[NOALLOC_MAX_DEVICES] = {};

static int noalloc_scratch_address(int device, unsigned char** out) {
    if (device < 0 || device >= NOALLOC_MAX_DEVICES) return fail(GN_INVALID_ARGUMENT, "gn_nav_compute_step_noalloc: device index beyond 63");
    std::lock_guard<std::mutex> lock(noalloc_mutex);
    if (!noalloc_ptr[device]) {
        unsigned char* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, noalloc_scratch);
        if (e != cudaSuccess || !p) { cudaGetLastError(); return cuda_fail(e, "gn_nav_compute_step_noalloc: cudaGetSymbolAddress"); }
        noalloc_ptr[device] = p;
    }
    *out = noalloc_ptr[device];
    return GN_OK;
}

// step_impl (nav_kernels.cuh) with the sort scratch in the static array
template <class R>
static int step_noalloc(const gn_geometry* geo, const void* pos, const void* dir, const int32_t* vol, const void* ms, int64_t n,
                        void* step, int32_t* next, cudaStream_t s) {
    if (n == 0) return GN_OK;
    if (geo->coherent) {                                                    // unrotated boxes only: no sort, no scratch
        step_kernel<R, false><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, (const R*)dir, vol, (const R*)ms, n, (R*)step, next, nullptr);
        GN_CUDA(cudaGetLastError(), "gn_nav_compute_step_noalloc launch");
        return GN_OK;
    }
    unsigned char* scratch = nullptr;
    const int rc = noalloc_scratch_address(geo->device, &scratch);
    if (rc != GN_OK) return rc;
    unsigned long long* totals = (unsigned long long*)scratch; unsigned long long* cursors = totals + SORT_KEYS_MAX;
    unsigned long long* totals2 = cursors + SORT_KEYS_MAX;
    uint8_t* keys = scratch + NOALLOC_HEAD;
    uint32_t* perm = (uint32_t*)(scratch + NOALLOC_HEAD + (size_t)NOALLOC_MAX_QUERIES);
    GN_CUDA(cudaMemsetAsync(scratch, 0, NOALLOC_HEAD, s), "gn_nav_compute_step_noalloc memset");      // the last call's counts
    sort_keys_kernel<R><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), vol, n, keys, totals);
    sort_scatter_kernel<<<nav_grid((n + 3) / 4), NAV_THREADS, 0, s>>>(keys, n, totals, cursors, perm, nullptr);
    step_two_wavefronts<R>(geo, pos, dir, vol, ms, n, step, next, perm, keys, totals2, s);
    GN_CUDA(cudaGetLastError(), "gn_nav_compute_step_noalloc launch");
    return GN_OK;
}

}  // namespace gn

using namespace gn;

extern "C" int gn_nav_compute_step_noalloc(const gn_geometry* geo, int precision, const void* d_pos, const void* d_dir,
                                           const int32_t* d_vol_in, const void* d_max_step, int64_t n, void* d_step_out,
                                           int32_t* d_next_vol_out, void* cuda_stream) {
    if (!geo || n < 0 || (n > 0 && (!d_pos || !d_dir || !d_vol_in || !d_step_out || !d_next_vol_out)))
        return fail(GN_INVALID_ARGUMENT, "gn_nav_compute_step_noalloc: bad argument");
    if (precision != 32 && precision != 64) return fail(GN_INVALID_ARGUMENT, "gn_nav_compute_step_noalloc: precision must be 32 or 64");
    if (n > NOALLOC_MAX_QUERIES)
        return fail(GN_INVALID_ARGUMENT, "gn_nav_compute_step_noalloc: n = " + std::to_string(n) + " exceeds GN_NOALLOC_MAX_QUERIES = " +
                                         std::to_string(NOALLOC_MAX_QUERIES) + " (the fixed scratch array); split the batch or call gn_nav_compute_step");
    // run on the geometry's device; the caller's current device is restored on return
    int prev = -1; bool switched = false;
    if (cudaGetDevice(&prev) == cudaSuccess && prev != geo->device) switched = cudaSetDevice(geo->device) == cudaSuccess;
    const cudaStream_t s = (cudaStream_t)cuda_stream;
    const int rc = precision == 32 ? step_noalloc<float>(geo, d_pos, d_dir, d_vol_in, d_max_step, n, d_step_out, d_next_vol_out, s)
                                   : step_noalloc<double>(geo, d_pos, d_dir, d_vol_in, d_max_step, n, d_step_out, d_next_vol_out, s);
    if (switched) cudaSetDevice(prev);
    return rc;
}
