// dr_static.cu -- dr_avg_stress_static (include/dr.h): the volume averages of Eq. 7 (Reading R7) for callers that
// cannot hand the library a workspace and cannot allocate one.
//
// Who that is.  Every other compute call of libdr works in a caller-owned workspace, which somebody had to cudaMalloc
// (or take from a framework's pool).  Two kinds of callers can do neither:
//   * a monitoring or post-processing hook that runs beside a long solve: cudaMalloc / cudaFree serialise against all work
//     on the device, so an allocation there stalls the solver's streams at every call;
//   * a plug-in inside a host application whose own allocator has already reserved the device memory that is left next to
//     a large image (the state of a 479^3 solve takes 19 GB, six load cases at once 111 GB): a cudaMalloc from the plug-in
//     fails, or succeeds only by starving the host.
// For them the scratch of the two-pass reduction lives in this library's own image: a file-scope __device__ array below,
// 6 MiB, present on every GPU that loads libdr.so for as long as the process lives.  The price is a size limit and no
// concurrency (see dr.h).
//
// The arithmetic is k_avg_partial / k_avg_final of dr_kernels_aux.cuh restated for DENSE fields (the arrays dr_get_field
// exports) instead of the padded boxes of a handle: plain cell sum for the normal stresses, trapezoid weights 1/2 on the first
// and last index of the two staggered directions of each edge shear.  One warp adds one x-row (j,k), a block adds its 8
// rows in a fixed order and writes 6 partial sums; the second kernel adds the partials in a fixed order -> the result
// does not depend on scheduling.  The grouping of the sum differs from dr_avg_stress, so the two agree to rounding
// (a few ulp of the largest component), not bit for bit.
//
// This file shares nothing with dr_api.cu but the public header: no existing call changes.
#include <cuda_runtime.h>
#include <cstdio>
#include <mutex>

#include "../../include/dr.h"

#define DRS_ROWS_PER_BLOCK 8                                  // one warp per row
#define DRS_THREADS (32 * DRS_ROWS_PER_BLOCK)
#define DRS_MAX_BLOCKS (DR_STATIC_MAX_ROWS / DRS_ROWS_PER_BLOCK)
#define DRS_MAX_DEVICES 64

// The scratch: 6 partial sums per block of the first pass.  In HOST code `drs_partial` is only the handle the runtime
// registered for this symbol -- NOT a device address; a kernel must be given the result of cudaGetSymbolAddress
// (drs_scratch_of below).  Device code may name it directly.
static __device__ __align__(256) double drs_partial[(size_t)DRS_MAX_BLOCKS * 6];

struct DrsFields { const double* f[6]; };                     // sxx, syy, szz, tyz, txz, txy (DEVICE, dense)

__device__ __forceinline__ double drs_warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// pass 1: block b adds the x-rows 8 b .. 8 b + 7 of the (ny+1) x (nz+1) node rows; partial[6 b + m]
__global__ void __launch_bounds__(DRS_THREADS)
k_avg_static_partial(int nx, int ny, int nz, DrsFields F, double* __restrict__ partial) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long rows = (long long)(ny + 1) * (nz + 1);
    const long long r = (long long)blockIdx.x * DRS_ROWS_PER_BLOCK + warp;
    double s[6] = {0, 0, 0, 0, 0, 0};
    if (r < rows) {
        const int k = (int)(r / (ny + 1)), j = (int)(r - (long long)k * (ny + 1));
        const bool cj = j < ny, ck = k < nz;
        const double wj = (j == 0 || j == ny) ? 0.5 : 1.0, wk = (k == 0 || k == nz) ? 0.5 : 1.0;
        const size_t X = (size_t)nx, X1 = (size_t)nx + 1, Y = (size_t)ny, Y1 = (size_t)ny + 1;
        const size_t qc = X * (j + Y * k);                    // cells      (nx,   ny,   nz)
        const size_t qyz = X * (j + Y1 * k);                  // tyz edges  (nx,   ny+1, nz+1)
        const size_t qxz = X1 * (j + Y * k);                  // txz edges  (nx+1, ny,   nz+1)
        const size_t qxy = X1 * (j + Y1 * k);                 // txy edges  (nx+1, ny+1, nz)
#pragma unroll 4
        for (int i = lane; i <= nx; i += 32) {
            const bool ci = i < nx;
            const double wi = (i == 0 || i == nx) ? 0.5 : 1.0;
            if (ci && cj && ck) { s[0] += F.f[0][qc + i]; s[1] += F.f[1][qc + i]; s[2] += F.f[2][qc + i]; }
            if (ci) s[3] += wj * wk * F.f[3][qyz + i];
            if (cj) s[4] += wi * wk * F.f[4][qxz + i];
            if (ck) s[5] += wi * wj * F.f[5][qxy + i];
        }
    }
    __shared__ double sm[6][DRS_ROWS_PER_BLOCK];
#pragma unroll
    for (int m = 0; m < 6; ++m) {
        const double v = drs_warp_sum(s[m]);
        if (lane == 0) sm[m][warp] = v;
    }
    __syncthreads();
    if (threadIdx.x < 6) {
        double v = 0;
        for (int w = 0; w < DRS_ROWS_PER_BLOCK; ++w) v += sm[threadIdx.x][w];
        partial[(size_t)blockIdx.x * 6 + threadIdx.x] = v;
    }
}

// pass 2 (one block): out6[m] = invN * sum over the nblocks partials this call wrote; entries beyond nblocks (left by an
// earlier, larger call) are never read
__global__ void __launch_bounds__(512)
k_avg_static_final(const double* __restrict__ partial, int nblocks, double invN, double* __restrict__ out6) {
    __shared__ double sm[6][512];
    double s[6] = {0, 0, 0, 0, 0, 0};
    for (int b = threadIdx.x; b < nblocks; b += 512)
        for (int m = 0; m < 6; ++m) s[m] += partial[(size_t)b * 6 + m];
    for (int m = 0; m < 6; ++m) sm[m][threadIdx.x] = s[m];
    __syncthreads();
    for (int o = 256; o > 0; o >>= 1) {
        if (threadIdx.x < o) for (int m = 0; m < 6; ++m) sm[m][threadIdx.x] += sm[m][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x < 6) out6[threadIdx.x] = sm[threadIdx.x][0] * invN;
}

// Device address of drs_partial on the CURRENT device, looked up once per device and process.  Each device that loads
// the library has its own copy of the array at its own address, hence the table; the lookup must run with that device
// current, which is why it sits here and not in a static initialiser.
static cudaError_t drs_scratch_of(int device, double** out) {
    static std::mutex mu;
    static double* addr[DRS_MAX_DEVICES] = {nullptr};
    std::lock_guard<std::mutex> lk(mu);
    if (!addr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, drs_partial);
        if (e != cudaSuccess) return e;
        addr[device] = (double*)p;
    }
    *out = addr[device];
    return cudaSuccess;
}

static dr_status drs_fail(dr_status s, char* errbuf, size_t n, const char* msg, const char* detail = nullptr) {
    if (errbuf && n) std::snprintf(errbuf, n, detail ? "%s: %s" : "%s", msg, detail);
    return s;
}

extern "C" dr_status dr_avg_stress_static(int nx, int ny, int nz, const double* const stress[6], double* out6,
                                          void* cuda_stream, char* errbuf, size_t errbuf_len) {
    if (errbuf && errbuf_len) errbuf[0] = 0;
    if (!stress || !out6) return drs_fail(DR_ERR_ARG, errbuf, errbuf_len, "dr_avg_stress_static: NULL stress[] or out6");
    for (int m = 0; m < 6; ++m)
        if (!stress[m]) return drs_fail(DR_ERR_ARG, errbuf, errbuf_len, "dr_avg_stress_static: NULL field pointer in stress[]");
    if (nx < 2 || ny < 2 || nz < 2 || nx > 8192 || ny > 8192 || nz > 8192)
        return drs_fail(DR_ERR_ARG, errbuf, errbuf_len, "dr_avg_stress_static: nx, ny, nz must lie in 2 .. 8192");
    const long long rows = (long long)(ny + 1) * (nz + 1);
    if (rows > (long long)DR_STATIC_MAX_ROWS) {
        if (errbuf && errbuf_len)
            std::snprintf(errbuf, errbuf_len,
                          "dr_avg_stress_static: (ny+1)*(nz+1) = %lld exceeds DR_STATIC_MAX_ROWS = %d, the size of the built-in "
                          "scratch; use dr_avg_stress on a handle (caller-owned workspace) for this grid", rows, (int)DR_STATIC_MAX_ROWS);
        return DR_ERR_ARG;
    }
    int device = -1;
    cudaError_t e = cudaGetDevice(&device);
    if (e != cudaSuccess) return drs_fail(DR_ERR_CUDA, errbuf, errbuf_len, "dr_avg_stress_static: cudaGetDevice", cudaGetErrorString(e));
    if (device < 0 || device >= DRS_MAX_DEVICES)
        return drs_fail(DR_ERR_CUDA, errbuf, errbuf_len, "dr_avg_stress_static: device ordinal beyond the 64 this call keeps an address for");
    double* scratch = nullptr;
    e = drs_scratch_of(device, &scratch);
    if (e != cudaSuccess) return drs_fail(DR_ERR_CUDA, errbuf, errbuf_len, "dr_avg_stress_static: cudaGetSymbolAddress", cudaGetErrorString(e));

    const cudaStream_t st = (cudaStream_t)cuda_stream;
    const int nblocks = (int)((rows + DRS_ROWS_PER_BLOCK - 1) / DRS_ROWS_PER_BLOCK);
    DrsFields F;
    for (int m = 0; m < 6; ++m) F.f[m] = stress[m];
    k_avg_static_partial<<<nblocks, DRS_THREADS, 0, st>>>(nx, ny, nz, F, scratch);
    e = cudaGetLastError();
    if (e != cudaSuccess) return drs_fail(DR_ERR_CUDA, errbuf, errbuf_len, "k_avg_static_partial", cudaGetErrorString(e));
    k_avg_static_final<<<1, 512, 0, st>>>(scratch, nblocks, 1.0 / ((double)nx * ny * nz), out6);
    e = cudaGetLastError();
    if (e != cudaSuccess) return drs_fail(DR_ERR_CUDA, errbuf, errbuf_len, "k_avg_static_final", cudaGetErrorString(e));
    return DR_OK;
}
