// api.cu -- the extern "C" entry points of include/gammanav.h: argument checks, precision / geometry-kind dispatch to the
// launchers (impl.h), the host-buffer wrappers (chunked, copies overlapped with kernels on two streams) and the device
// self-tests (correctly rounded in-line division / square root; FP32 / FP64 pipe peak).
#include <cmath>
#include "common.cuh"
#include "hostmath.h"
#include "impl.h"
#include "physics.cuh"

namespace gn {

// Every entry point runs on the device the geometry was created on (its pointers live there); the caller's current
// device is restored on return.
struct DeviceScope {
    int prev = -1; bool switched = false;
    explicit DeviceScope(const gn_geometry* geo) {
        if (cudaGetDevice(&prev) == cudaSuccess && geo && prev != geo->device) switched = cudaSetDevice(geo->device) == cudaSuccess;
    }
    ~DeviceScope() { if (switched) cudaSetDevice(prev); }
};

// Device form of the photon source: the frame comes from hostmath.h in fp64
// and is rounded once to Real.
template <class R> bool make_source(const gn_source& s, SourceDev<R>& o) {
    const bool mono = s.energy_kind == GN_E_MONO, loguni = s.energy_kind == GN_E_LOGUNIFORM;
    if (s.kind < GN_SRC_PENCIL || s.kind > GN_SRC_ISOTROPIC || !(mono || loguni) || !(s.e0 > 0)) return false;
    if (loguni && !(s.e1 >= s.e0)) return false;
    SourceFrame f;
    if (!source_frame(s.axis, f)) return false;
    o.kind = s.kind; o.energy_kind = s.energy_kind;
    o.o[0] = (R)s.origin[0]; o.o[1] = (R)s.origin[1]; o.o[2] = (R)s.origin[2];
    o.a[0] = (R)f.a.x; o.a[1] = (R)f.a.y; o.a[2] = (R)f.a.z;
    o.e1[0] = (R)f.e1.x; o.e1[1] = (R)f.e1.y; o.e1[2] = (R)f.e1.z;
    o.e2[0] = (R)f.e2.x; o.e2[1] = (R)f.e2.y; o.e2[2] = (R)f.e2.z;
    o.sigma = (R)s.sigma;
    o.cos_half = (R)std::cos(s.half_angle);
    o.e0 = (R)s.e0;
    o.ln_e0 = loguni ? (R)std::log(s.e0) : (R)0;
    o.ln_ratio = loguni ? (R)std::log(s.e1 / s.e0) : (R)0;
    return true;
}

template <class R>
static int transport_dispatch(const gn_geometry* geo, const gn_source* h_src, uint64_t seed, int64_t first_id, int64_t n, double* d_edep,
                              gn_run_stats* h_stats, uint64_t* d_hash, uint32_t* d_nsteps, double* d_efinal, cudaStream_t s) {
    SourceDev<R> src;
    if (!make_source(*h_src, src)) return fail(GN_INVALID_ARGUMENT, "gn_transport_run: bad source (axis, energies or kind)");
    if (geo->coherent) return transport_impl<R, false>(geo, src, seed, first_id, n, d_edep, h_stats, d_hash, d_nsteps, d_efinal, s);
    return transport_impl<R, true>(geo, src, seed, first_id, n, d_edep, h_stats, d_hash, d_nsteps, d_efinal, s);
}

}  // namespace gn

using namespace gn;

extern "C" int gn_nav_locate(const gn_geometry* geo, int precision, const void* d_pos, const void* d_dir, int64_t n,
                             int32_t* d_vol_out, void* cuda_stream) {
    if (!geo || n < 0 || (n > 0 && (!d_pos || !d_vol_out))) return fail(GN_INVALID_ARGUMENT, "gn_nav_locate: bad argument");
    DeviceScope dev(geo);
    if (precision == 32) return locate_impl<float>(geo, d_pos, d_dir, n, d_vol_out, (cudaStream_t)cuda_stream);
    if (precision == 64) return locate_impl<double>(geo, d_pos, d_dir, n, d_vol_out, (cudaStream_t)cuda_stream);
    return fail(GN_INVALID_ARGUMENT, "gn_nav_locate: precision must be 32 or 64");
}

extern "C" int gn_nav_compute_step(const gn_geometry* geo, int precision, const void* d_pos, const void* d_dir,
                                   const int32_t* d_vol_in, const void* d_max_step, int64_t n, void* d_step_out,
                                   int32_t* d_next_vol_out, void* cuda_stream) {
    if (!geo || n < 0 || (n > 0 && (!d_pos || !d_dir || !d_vol_in || !d_step_out || !d_next_vol_out)))
        return fail(GN_INVALID_ARGUMENT, "gn_nav_compute_step: bad argument");
    DeviceScope dev(geo);
    if (precision == 32) return step_impl<float>(geo, d_pos, d_dir, d_vol_in, d_max_step, n, d_step_out, d_next_vol_out, (cudaStream_t)cuda_stream);
    if (precision == 64) return step_impl<double>(geo, d_pos, d_dir, d_vol_in, d_max_step, n, d_step_out, d_next_vol_out, (cudaStream_t)cuda_stream);
    return fail(GN_INVALID_ARGUMENT, "gn_nav_compute_step: precision must be 32 or 64");
}

extern "C" int gn_nav_compute_step_normal(const gn_geometry* geo, int precision, const void* d_pos, const void* d_dir, const int32_t* d_vol_in,
                                          const void* d_max_step, int64_t n, void* d_step_out, int32_t* d_next_vol_out, void* d_normal_out,
                                          void* cuda_stream) {
    if (!geo || n < 0 || (n > 0 && (!d_pos || !d_dir || !d_vol_in || !d_step_out || !d_next_vol_out || !d_normal_out)))
        return fail(GN_INVALID_ARGUMENT, "gn_nav_compute_step_normal: bad argument");
    DeviceScope dev(geo);
    if (precision == 32) return step_normal_impl<float>(geo, d_pos, d_dir, d_vol_in, d_max_step, n, d_step_out, d_next_vol_out, d_normal_out, (cudaStream_t)cuda_stream);
    if (precision == 64) return step_normal_impl<double>(geo, d_pos, d_dir, d_vol_in, d_max_step, n, d_step_out, d_next_vol_out, d_normal_out, (cudaStream_t)cuda_stream);
    return fail(GN_INVALID_ARGUMENT, "gn_nav_compute_step_normal: precision must be 32 or 64");
}

extern "C" int gn_nav_compute_safety(const gn_geometry* geo, int precision, const void* d_pos, const int32_t* d_vol_in, int64_t n,
                                     void* d_safety_out, void* cuda_stream) {
    if (!geo || n < 0 || (n > 0 && (!d_pos || !d_vol_in || !d_safety_out))) return fail(GN_INVALID_ARGUMENT, "gn_nav_compute_safety: bad argument");
    DeviceScope dev(geo);
    if (precision == 32) return safety_impl<float>(geo, d_pos, d_vol_in, n, d_safety_out, (cudaStream_t)cuda_stream);
    if (precision == 64) return safety_impl<double>(geo, d_pos, d_vol_in, n, d_safety_out, (cudaStream_t)cuda_stream);
    return fail(GN_INVALID_ARGUMENT, "gn_nav_compute_safety: precision must be 32 or 64");
}

extern "C" int gn_transport_run(const gn_geometry* geo, int precision, const gn_source* h_src, uint64_t seed, int64_t first_photon_id,
                                int64_t n_photons, double* d_edep_out, gn_run_stats* h_stats_out, uint64_t* d_hash_out,
                                uint32_t* d_nsteps_out, double* d_efinal_out, void* cuda_stream) {
    if (!geo || !h_src || !d_edep_out || n_photons < 0 || first_photon_id < 0) return fail(GN_INVALID_ARGUMENT, "gn_transport_run: bad argument");
    if (h_stats_out) std::memset(h_stats_out, 0, sizeof *h_stats_out);
    DeviceScope dev(geo);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (precision == 32) return transport_dispatch<float>(geo, h_src, seed, first_photon_id, n_photons, d_edep_out, h_stats_out, d_hash_out, d_nsteps_out, d_efinal_out, s);
    if (precision == 64) return transport_dispatch<double>(geo, h_src, seed, first_photon_id, n_photons, d_edep_out, h_stats_out, d_hash_out, d_nsteps_out, d_efinal_out, s);
    return fail(GN_INVALID_ARGUMENT, "gn_transport_run: precision must be 32 or 64");
}

extern "C" int gn_free_path_run(const gn_geometry* geo, int precision, const void* d_pos, const void* d_dir, const void* d_Y, int64_t n,
                                double mu_mass_cm2_g, void* d_T_out, uint32_t* d_nsteps_out, void* cuda_stream) {
    if (!geo || n < 0 || !(mu_mass_cm2_g >= 0) || (n > 0 && (!d_pos || !d_dir || !d_Y || !d_T_out)))
        return fail(GN_INVALID_ARGUMENT, "gn_free_path_run: bad argument");
    DeviceScope dev(geo);
    if (precision == 32) return free_path_impl<float>(geo, d_pos, d_dir, d_Y, n, mu_mass_cm2_g, d_T_out, d_nsteps_out, (cudaStream_t)cuda_stream);
    if (precision == 64) return free_path_impl<double>(geo, d_pos, d_dir, d_Y, n, mu_mass_cm2_g, d_T_out, d_nsteps_out, (cudaStream_t)cuda_stream);
    return fail(GN_INVALID_ARGUMENT, "gn_free_path_run: precision must be 32 or 64");
}

// -------------------------------------------------------------------------------------------------------
// host-buffer entry points: the query arrays are cut into chunks; chunk c uses stream c % 2 and its own half of a
// device staging area owned by the handle, so the upload of chunk c + 1 and the download of chunk c - 1 overlap the
// kernels of chunk c (needs page-locked caller buffers to overlap; pageable ones are copied correctly but serially)
// -------------------------------------------------------------------------------------------------------
namespace gn {
constexpr int64_t HOST_CHUNK = 1ll << 22;          // queries per chunk

static int host_pipe_prepare(const gn_geometry* geo, size_t bytes_per_slot) {
    if (!geo->hp_streams_ok) {
        bool ok = true;
        for (int k = 0; k < 2; ++k) ok = ok && cudaStreamCreateWithFlags(&geo->hp_stream[k], cudaStreamNonBlocking) == cudaSuccess;
        if (!ok) { cudaGetLastError(); return fail(GN_CUDA_ERROR, "host pipe: stream create"); }
        geo->hp_streams_ok = true;
    }
    if (geo->hp_bytes < 2 * bytes_per_slot) {
        if (geo->hp_buf) { cudaDeviceSynchronize(); cudaFree(geo->hp_buf); geo->hp_buf = nullptr; geo->hp_bytes = 0; }
        if (cudaMalloc((void**)&geo->hp_buf, 2 * bytes_per_slot) != cudaSuccess) { cudaGetLastError(); geo->hp_buf = nullptr; return fail(GN_OUT_OF_MEMORY, "host pipe: cudaMalloc"); }
        geo->hp_bytes = 2 * bytes_per_slot;
    }
    return GN_OK;
}
}  // namespace gn

extern "C" int gn_nav_query_host(const gn_geometry* geo, int precision, const void* h_pos, const void* h_dir, int64_t n,
                                 int32_t* h_vol_out, void* h_step_out, int32_t* h_next_vol_out) {
    if (!geo || n < 0 || (precision != 32 && precision != 64) || (n > 0 && (!h_pos || !h_dir || !h_vol_out || !h_step_out || !h_next_vol_out)))
        return fail(GN_INVALID_ARGUMENT, "gn_nav_query_host: bad argument");
    if (n == 0) return GN_OK;
    DeviceScope dev(geo);
    std::lock_guard<std::mutex> host_lock(geo->host_mutex);
    const size_t rs = precision == 32 ? 4 : 8;
    const int64_t chunk = std::min<int64_t>(n, HOST_CHUNK);
    const size_t b_pos = 3 * rs * (size_t)chunk, b_i = 4 * (size_t)chunk, b_r = rs * (size_t)chunk;
    const size_t slot = (2 * b_pos + 2 * b_i + b_r + 255) & ~(size_t)255;
    int rc = host_pipe_prepare(geo, slot);
    if (rc != GN_OK) return rc;
    cudaError_t e = cudaSuccess;
    for (int64_t off = 0, c = 0; off < n && rc == GN_OK && e == cudaSuccess; off += chunk, ++c) {
        const int64_t m = std::min(chunk, n - off);
        cudaStream_t s = geo->hp_stream[c & 1];
        char* d = geo->hp_buf + (c & 1) * slot;
        char *dp = d, *dd = d + b_pos, *dstep = d + 2 * b_pos, *dvol = dstep + b_r, *dnext = dvol + b_i;
        e = cudaMemcpyAsync(dp, (const char*)h_pos + 3 * rs * (size_t)off, 3 * rs * (size_t)m, cudaMemcpyHostToDevice, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(dd, (const char*)h_dir + 3 * rs * (size_t)off, 3 * rs * (size_t)m, cudaMemcpyHostToDevice, s);
        if (e != cudaSuccess) break;
        rc = gn_nav_locate(geo, precision, dp, dd, m, (int32_t*)dvol, s);
        if (rc == GN_OK) rc = gn_nav_compute_step(geo, precision, dp, dd, (const int32_t*)dvol, nullptr, m, dstep, (int32_t*)dnext, s);
        if (rc != GN_OK) break;
        e = cudaMemcpyAsync(h_vol_out + off, dvol, 4 * (size_t)m, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync((char*)h_step_out + rs * (size_t)off, dstep, rs * (size_t)m, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(h_next_vol_out + off, dnext, 4 * (size_t)m, cudaMemcpyDeviceToHost, s);
    }
    for (int k = 0; k < 2; ++k) { cudaError_t e2 = cudaStreamSynchronize(geo->hp_stream[k]); if (e == cudaSuccess) e = e2; }
    if (rc != GN_OK) return rc;
    if (e != cudaSuccess) return cuda_fail(e, "gn_nav_query_host");
    return GN_OK;
}

extern "C" int gn_free_path_run_host(const gn_geometry* geo, int precision, const void* h_pos, const void* h_dir, const void* h_Y, int64_t n,
                                     double mu_mass_cm2_g, void* h_T_out, uint32_t* h_nsteps_out) {
    if (!geo || n < 0 || (precision != 32 && precision != 64) || (n > 0 && (!h_pos || !h_dir || !h_Y || !h_T_out)))
        return fail(GN_INVALID_ARGUMENT, "gn_free_path_run_host: bad argument");
    if (n == 0) return GN_OK;
    DeviceScope dev(geo);
    std::lock_guard<std::mutex> host_lock(geo->host_mutex);
    const size_t rs = precision == 32 ? 4 : 8;
    const int64_t chunk = std::min<int64_t>(n, HOST_CHUNK);
    const size_t b3 = 3 * rs * (size_t)chunk, b1 = rs * (size_t)chunk, bi = 4 * (size_t)chunk;
    const size_t slot = (2 * b3 + 2 * b1 + bi + 255) & ~(size_t)255;
    int rc = host_pipe_prepare(geo, slot);
    if (rc != GN_OK) return rc;
    cudaError_t e = cudaSuccess;
    // Algorithm 2 phases 4-6: transfer the particle states and lifetimes, compute, transfer T back
    for (int64_t off = 0, c = 0; off < n && rc == GN_OK && e == cudaSuccess; off += chunk, ++c) {
        const int64_t m = std::min(chunk, n - off);
        cudaStream_t s = geo->hp_stream[c & 1];
        char* d = geo->hp_buf + (c & 1) * slot;
        char *dp = d, *dd = d + b3, *dY = d + 2 * b3, *dT = dY + b1, *dn = dT + b1;
        e = cudaMemcpyAsync(dp, (const char*)h_pos + 3 * rs * (size_t)off, 3 * rs * (size_t)m, cudaMemcpyHostToDevice, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(dd, (const char*)h_dir + 3 * rs * (size_t)off, 3 * rs * (size_t)m, cudaMemcpyHostToDevice, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(dY, (const char*)h_Y + rs * (size_t)off, rs * (size_t)m, cudaMemcpyHostToDevice, s);
        if (e != cudaSuccess) break;
        rc = gn_free_path_run(geo, precision, dp, dd, dY, m, mu_mass_cm2_g, dT, h_nsteps_out ? (uint32_t*)dn : nullptr, s);
        if (rc != GN_OK) break;
        e = cudaMemcpyAsync((char*)h_T_out + rs * (size_t)off, dT, rs * (size_t)m, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess && h_nsteps_out) e = cudaMemcpyAsync(h_nsteps_out + off, dn, 4 * (size_t)m, cudaMemcpyDeviceToHost, s);
    }
    for (int k = 0; k < 2; ++k) { cudaError_t e2 = cudaStreamSynchronize(geo->hp_stream[k]); if (e == cudaSuccess) e = e2; }
    if (rc != GN_OK) return rc;
    if (e != cudaSuccess) return cuda_fail(e, "gn_free_path_run_host");
    return GN_OK;
}

extern "C" int gn_transport_run_host(const gn_geometry* geo, int precision, const gn_source* h_src, uint64_t seed,
                                     int64_t first_photon_id, int64_t n_photons, double* h_edep_out, gn_run_stats* h_stats_out) {
    if (!geo || !h_edep_out) return fail(GN_INVALID_ARGUMENT, "gn_transport_run_host: bad argument");
    DeviceScope dev(geo);
    const size_t bytes = sizeof(double) * (size_t)geo->n_places;
    double* d = nullptr;
    std::lock_guard<std::mutex> host_lock(geo->host_mutex);
    {   // the device staging buffer of the tally belongs to the handle (no allocation per call)
        if (!geo->ws_host_edep && cudaMalloc((void**)&geo->ws_host_edep, bytes) != cudaSuccess) {
            cudaGetLastError(); geo->ws_host_edep = nullptr;
            return fail(GN_OUT_OF_MEMORY, "gn_transport_run_host: cudaMalloc");
        }
        d = geo->ws_host_edep;
    }
    int rc = gn_transport_run(geo, precision, h_src, seed, first_photon_id, n_photons, d, h_stats_out, nullptr, nullptr, nullptr, nullptr);
    if (rc != GN_OK) return rc;
    cudaError_t e = cudaMemcpy(h_edep_out, d, bytes, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(e, "gn_transport_run_host");
    return GN_OK;
}

// host-only hooks (no device needed): the set-up arithmetic of the library, for tests that compare it with an independent
// implementation of the same definitions
extern "C" int gn_host_source_frame(const gn_source* h_src, int precision, double frame_out[9]) {
    if (!h_src || !frame_out || (precision != 32 && precision != 64)) return fail(GN_INVALID_ARGUMENT, "gn_host_source_frame: bad argument");
    if (precision == 32) {
        SourceDev<float> s;
        if (!make_source(*h_src, s)) return fail(GN_INVALID_ARGUMENT, "gn_host_source_frame: bad source");
        for (int i = 0; i < 3; ++i) { frame_out[i] = s.a[i]; frame_out[3 + i] = s.e1[i]; frame_out[6 + i] = s.e2[i]; }
    } else {
        SourceDev<double> s;
        if (!make_source(*h_src, s)) return fail(GN_INVALID_ARGUMENT, "gn_host_source_frame: bad source");
        for (int i = 0; i < 3; ++i) { frame_out[i] = s.a[i]; frame_out[3 + i] = s.e1[i]; frame_out[6 + i] = s.e2[i]; }
    }
    return GN_OK;
}

// -------------------------------------------------------------------------------------------------------
// arithmetic self-test: the in-line correctly rounded fp32 division / square root of nav.cuh against the
// toolchain's __fdiv_rn / __fsqrt_rn (IEEE round-to-nearest), bit for bit
// -------------------------------------------------------------------------------------------------------
namespace gn {
__device__ __forceinline__ uint32_t mix32(uint64_t z) {          // splitmix64 finaliser
    z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ull; z = (z ^ (z >> 27)) * 0x94d049bb133111ebull; z ^= z >> 31;
    return (uint32_t)(z >> 16);
}
__global__ void selftest_sqrt_kernel(unsigned long long* out) {
    unsigned bad = 0;
    for (uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; i < (1ull << 32); i += (uint64_t)gridDim.x * blockDim.x) {
        float a = __uint_as_float((uint32_t)i);
        float mine = rsqrt_(a), ref = __fsqrt_rn(a);
        bool same = __float_as_uint(mine) == __float_as_uint(ref) || (mine != mine && ref != ref);
        if (!same) { ++bad; atomicMin(&out[2], (unsigned long long)i); }
    }
    if (bad) atomicAdd(&out[0], (unsigned long long)bad);
}
__global__ void selftest_div_kernel(unsigned long long n, unsigned long long* out) {
    unsigned bad = 0;
    for (uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
        uint32_t ua = mix32(2 * i + 1), ub = mix32(2 * i + 2) ^ 0x9e3779b9u;
        const unsigned mode = (unsigned)(i & 3);
        if (mode == 1) {                      // exponents of lengths and direction cosines: 2^-24 .. 2^16
            ua = (ua & 0x807fffffu) | ((103u + (ua >> 23) % 40u) << 23); ub = (ub & 0x807fffffu) | ((103u + (ub >> 23) % 40u) << 23);
        } else if (mode == 2) {               // quotient just below / above a power of two and a rounding boundary
            ub = (ub & 0x807fffffu) | (127u << 23); ua = (ua & 0x80000000u) | ((ub & 0x7fffffffu) + (ua & 3u) - 1u);
        } else if (mode == 3) {               // few mantissa bits: exact and half-way cases
            ua &= 0xfff80000u; ub &= 0xffe00000u;
        }
        float a = __uint_as_float(ua), b = __uint_as_float(ub);
        float mine = rdiv(a, b), ref = __fdiv_rn(a, b);
        bool same = __float_as_uint(mine) == __float_as_uint(ref) || (mine != mine && ref != ref);
        // the cached-reciprocal form used by the regular-voxel step (nav.cuh: RcpDir) must give the same bits whenever it is used
        if (mid_range(a) && mid_range(b)) {
            const float r = refined_rcp(b);
            same = same && __float_as_uint(div_by_rcp(a, b, r)) == __float_as_uint(ref);
        }
        const float ar = fabsf(ref);
        if (!same && ar < 1.17549435e-38f) same = fabsf(mine) < 1.17549435e-38f * 1.0001f;      // subnormal quotients: out of contract
        if (!same) { ++bad; atomicMin(&out[3], (unsigned long long)i); }
    }
    if (bad) atomicAdd(&out[1], (unsigned long long)bad);
}

// FP32 / FP64 pipe peak ("an FFMA / DFMA register-resident microbenchmark at the clock observed during the
// run"): every thread keeps 8 independent accumulator chains in registers and issues nothing but fused multiply-adds.
template <class R> __device__ __forceinline__ R pk_fma(R a, R b, R c);
template <> __device__ __forceinline__ float pk_fma<float>(float a, float b, float c) { return __fmaf_rn(a, b, c); }
template <> __device__ __forceinline__ double pk_fma<double>(double a, double b, double c) { return __fma_rn(a, b, c); }
template <class R> __global__ void __launch_bounds__(1024) pipe_peak_kernel(int iters, R seed, R* sink, long long* cycles) {
    R a0 = seed, a1 = seed + (R)1, a2 = seed + (R)2, a3 = seed + (R)3, a4 = seed + (R)4, a5 = seed + (R)5, a6 = seed + (R)6, a7 = seed + (R)7;
    const R m = (R)0.999, c = (R)threadIdx.x * (R)1e-6;
    const long long t0 = clock64();
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            a0 = pk_fma(a0, m, c); a1 = pk_fma(a1, m, c); a2 = pk_fma(a2, m, c); a3 = pk_fma(a3, m, c);
            a4 = pk_fma(a4, m, c); a5 = pk_fma(a5, m, c); a6 = pk_fma(a6, m, c); a7 = pk_fma(a7, m, c);
        }
    }
    const long long t1 = clock64();
    const R sum = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (sum == (R)-12345.678) sink[0] = sum;                          // never true: keeps the chains alive
    if (blockIdx.x == 0 && threadIdx.x == 0) cycles[0] = t1 - t0;
}
template <class R> int pipe_peak(double out[4]) {
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    char* d = nullptr;
    if (cudaMalloc((void**)&d, 64) != cudaSuccess) { cudaGetLastError(); return fail(GN_OUT_OF_MEMORY, "gn_selftest_pipe_peak: cudaMalloc"); }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = sms, threads = 1024;                           // one block per SM (its cycle count spans the kernel): 8 warps of 8 independent chains per scheduler
    const int iters = sizeof(R) == 4 ? 40000 : 8000;
    float best_ms = 1e30f; long long cyc = 0;
    for (int rep = 0; rep < 4; ++rep) {                               // first repetition warms the clocks up
        cudaEventRecord(e0);
        pipe_peak_kernel<R><<<blocks, threads>>>(iters, (R)(1.0 + rep), (R*)d, (long long*)(d + 32));
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best_ms) { best_ms = ms; cudaMemcpy(&cyc, d + 32, 8, cudaMemcpyDeviceToHost); }
    }
    cudaError_t e = cudaGetLastError();
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    if (e != cudaSuccess || !(best_ms < 1e29f)) return cuda_fail(e, "gn_selftest_pipe_peak");
    const double flops = 2.0 * 64.0 * (double)iters * (double)blocks * threads;      // 64 fma per iteration, 2 flops each
    out[0] = flops / (best_ms * 1e-3) / 1e12;                                        // TFLOP/s
    out[1] = (double)cyc / (best_ms * 1e-3) / 1e6;                                   // SM clock during the run [MHz] (block 0's cycle count / kernel time)
    out[2] = best_ms;
    out[3] = sms;
    return GN_OK;
}
}  // namespace gn

extern "C" int gn_selftest_arith(int64_t n_div_pairs, uint64_t h_out[4]) {
    if (!h_out || n_div_pairs < 0) return fail(GN_INVALID_ARGUMENT, "gn_selftest_arith: bad argument");
    unsigned long long* d = nullptr;
    if (cudaMalloc((void**)&d, 32) != cudaSuccess) { cudaGetLastError(); return fail(GN_OUT_OF_MEMORY, "gn_selftest_arith: cudaMalloc"); }
    unsigned long long init[4] = {0, 0, ~0ull, ~0ull};
    cudaMemcpy(d, init, 32, cudaMemcpyHostToDevice);
    selftest_sqrt_kernel<<<148 * 16, 256>>>(d);
    if (n_div_pairs > 0) selftest_div_kernel<<<148 * 16, 256>>>((unsigned long long)n_div_pairs, d);
    cudaError_t e = cudaMemcpy(h_out, d, 32, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return cuda_fail(e, "gn_selftest_arith");
    return GN_OK;
}

extern "C" int gn_selftest_pipe_peak(int precision, double h_out[4]) {
    if (!h_out || (precision != 32 && precision != 64)) return fail(GN_INVALID_ARGUMENT, "gn_selftest_pipe_peak: bad argument");
    int n = 0;
    if (cudaGetDeviceCount(&n) != cudaSuccess || n == 0) { cudaGetLastError(); return fail(GN_CUDA_ERROR, "gn_selftest_pipe_peak: no CUDA device"); }
    return precision == 32 ? pipe_peak<float>(h_out) : pipe_peak<double>(h_out);
}
