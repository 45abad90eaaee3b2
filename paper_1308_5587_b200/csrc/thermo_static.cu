// hb_thermo_static: the thermodynamic sums of hb_thermo for callers that must not allocate
// device memory.  Same two-stage binary64 reduction as thermo_partial_kernel / thermo_final_kernel of nve.cu, but
//   - it takes plain caller-owned device arrays (the layouts hb_get_state / hb_get_mass / hb_get_forces write),
//     no handle: hb_create allocates, so a handle is exactly what such a caller cannot make;
//   - the per-block partial sums, the only memory the reduction needs beyond its inputs and its output, live in a
//     fixed array inside the library image instead of a buffer obtained from cudaMalloc.
// Nothing here calls cudaMalloc, cudaFree, a stream-ordered allocator or a library routine that allocates.
//
// The array below costs SCRATCH_BYTES (360,448 B) of device memory on every GPU on which this library's module gets
// loaded, from that moment until the process exits, whether or not hb_thermo_static is ever called there.
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/hb.h"

namespace {

constexpr int TS_VALS = 11;         // K, U, W[6], px, py, pz  (the order of the partial sums)
constexpr int TS_THREADS = 256;
constexpr int TS_PER_THREAD = 16;
constexpr int TS_PER_BLOCK = TS_THREADS * TS_PER_THREAD;                                   // 4096 particles per block
constexpr int TS_MAX_BLOCKS = (int)(HB_THERMO_STATIC_MAX_N / TS_PER_BLOCK);                // 4096
constexpr size_t SCRATCH_BYTES = sizeof(double) * (size_t)TS_MAX_BLOCKS * TS_VALS;         // 360,448
static_assert((int64_t)TS_MAX_BLOCKS * TS_PER_BLOCK == HB_THERMO_STATIC_MAX_N, "the limit is a whole number of blocks");
static_assert(SCRATCH_BYTES == 360448, "hb.h and README.md state this figure");
constexpr int MAX_DEVICES = 64;

// One block's 11 partial sums at [block][TS_VALS].  In HOST code this name is only a handle for the runtime's symbol
// calls: it is not a device address, and a kernel handed `g_scratch` itself would fault (or, on a system where the
// GPU can reach host memory, quietly read and write the wrong bytes).  Host code gets the real address, per device,
// from cudaGetSymbolAddress (scratch_of_current_device below).
static __device__ __align__(256) double g_scratch[(size_t)TS_MAX_BLOCKS * TS_VALS];

// Block b sums particles [b * 4096, (b + 1) * 4096): which particles meet in which partial sum depends on N alone,
// not on the GPU, so the result is the same bit for bit wherever it runs.
__global__ void __launch_bounds__(TS_THREADS)
thermo_static_partial_kernel(const float *__restrict__ vel_xyz, const float *__restrict__ mass,
                             const float *__restrict__ f_xyz_u, const float *__restrict__ virial6, int64_t N,
                             double *__restrict__ part)
{
    double a[TS_VALS];
#pragma unroll
    for (int q = 0; q < TS_VALS; q++) a[q] = 0.0;
    const int64_t base = (int64_t)blockIdx.x * TS_PER_BLOCK;
    for (int k = 0; k < TS_PER_THREAD; k++) {
        const int64_t i = base + (int64_t)k * TS_THREADS + threadIdx.x;
        if (i >= N) break;
        const double m = mass ? (double)mass[i] : 1.0;
        const double vx = vel_xyz[3 * i], vy = vel_xyz[3 * i + 1], vz = vel_xyz[3 * i + 2];
        a[0] += 0.5 * m * (vx * vx + vy * vy + vz * vz);
        if (f_xyz_u) a[1] += (double)f_xyz_u[4 * i + 3];
        if (virial6) {
#pragma unroll
            for (int c = 0; c < 6; c++) a[2 + c] += (double)virial6[6 * i + c];
        }
        a[8] += m * vx; a[9] += m * vy; a[10] += m * vz;
    }
    __shared__ double sm[TS_THREADS / 32][TS_VALS];
#pragma unroll
    for (int q = 0; q < TS_VALS; q++) {
        double x = a[q];
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5][q] = x;
    }
    __syncthreads();
    if (threadIdx.x < TS_VALS) {
        double x = 0.0;
        for (int w = 0; w < TS_THREADS / 32; w++) x += sm[w][threadIdx.x];
        part[(int64_t)blockIdx.x * TS_VALS + threadIdx.x] = x;
    }
}

// One block of 11 warps: warp q adds up value q of every block in a fixed order, thread 0 then fills the hb_thermo_t.
__global__ void __launch_bounds__(TS_VALS * 32)
thermo_static_final_kernel(const double *__restrict__ part, int nblocks, double volume, double *__restrict__ out12)
{
    __shared__ double tot[TS_VALS];
    const int q = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double x = 0.0;
    for (int b = lane; b < nblocks; b += 32) x += part[(int64_t)b * TS_VALS + q];
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    if (lane == 0) tot[q] = x;
    __syncthreads();
    if (threadIdx.x == 0) {     // hb_thermo_t: K, U, W[6], P, px, py, pz
        out12[0] = tot[0];
        out12[1] = tot[1];
        for (int c = 0; c < 6; c++) out12[2 + c] = tot[2 + c];
        out12[8] = (2.0 * tot[0] + tot[2] + tot[5] + tot[7]) / (3.0 * volume);
        out12[9] = tot[8]; out12[10] = tot[9]; out12[11] = tot[10];
    }
}

int fail(char *errbuf, size_t errbuf_len, int code, const char *fmt, ...)
{
    if (errbuf && errbuf_len) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errbuf, errbuf_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// The device address of g_scratch on the CURRENT device, looked up once per device and then remembered.  Each GPU
// holds its own copy of the array, at its own address, so the answer of one device must never be used on another.
int scratch_of_current_device(double **out, char *errbuf, size_t errbuf_len)
{
    static std::mutex mu;
    static double *known[MAX_DEVICES] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(errbuf, errbuf_len, HB_ECUDA, "hb_thermo_static: cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= MAX_DEVICES)
        return fail(errbuf, errbuf_len, HB_EINVAL, "hb_thermo_static: device ordinal %d is outside 0..%d", dev, MAX_DEVICES - 1);
    std::lock_guard<std::mutex> lock(mu);
    if (!known[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return fail(errbuf, errbuf_len, HB_ECUDA, "hb_thermo_static: cudaGetSymbolAddress(scratch) on device %d: %s", dev,
                        cudaGetErrorString(e));
        }
        known[dev] = static_cast<double *>(p);
    }
    *out = known[dev];
    return HB_OK;
}

}  // namespace

extern "C" int hb_thermo_static(const float *vel_xyz, const float *mass, const float *f_xyz_u, const float *virial6,
                                int64_t N, double L, hb_thermo_t *out_device, void *cuda_stream, char *errbuf,
                                size_t errbuf_len)
{
    if (errbuf && errbuf_len) errbuf[0] = 0;
    if (!vel_xyz || !out_device) return fail(errbuf, errbuf_len, HB_EINVAL, "hb_thermo_static: vel_xyz and out_device must not be NULL");
    if (N <= 0) return fail(errbuf, errbuf_len, HB_EINVAL, "hb_thermo_static: N = %lld, need N >= 1", (long long)N);
    if (N > HB_THERMO_STATIC_MAX_N)
        return fail(errbuf, errbuf_len, HB_EINVAL,
                    "hb_thermo_static: N = %lld is more than HB_THERMO_STATIC_MAX_N = %lld particles, the most the fixed "
                    "scratch array holds partial sums for; use hb_thermo (which allocates) or split the particles over calls",
                    (long long)N, (long long)HB_THERMO_STATIC_MAX_N);
    if (!(L > 0.0)) return fail(errbuf, errbuf_len, HB_EINVAL, "hb_thermo_static: L = %g, need L > 0", L);
    double *scratch = nullptr;
    const int rc = scratch_of_current_device(&scratch, errbuf, errbuf_len);
    if (rc != HB_OK) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int nblocks = (int)((N + TS_PER_BLOCK - 1) / TS_PER_BLOCK);
    // Every partial sum the second kernel reads is written by the first in this same call: the contents a previous
    // call left in the array are never read, so there is nothing to clear.
    thermo_static_partial_kernel<<<nblocks, TS_THREADS, 0, stream>>>(vel_xyz, mass, f_xyz_u, virial6, N, scratch);
    thermo_static_final_kernel<<<1, TS_VALS * 32, 0, stream>>>(scratch, nblocks, L * L * L, reinterpret_cast<double *>(out_device));
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(errbuf, errbuf_len, HB_ECUDA, "hb_thermo_static: kernel launch: %s", cudaGetErrorString(e));
    return HB_OK;
}
