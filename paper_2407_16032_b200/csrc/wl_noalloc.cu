// wl_noalloc.cu -- wl_energy_static (include/wl.h): kinetic energy and enstrophy of a velocity field for callers that cannot
// allocate (code under CUDA-graph capture, serving loops, harnesses that forbid cudaMalloc).  A variant of k_energy (wl_flow.cu;
// PAPER.md:169-173, reading R-E2 of DESIGN.md) whose reduction scratch -- one pair of fp64 partial sums per block and the ticket
// counter that elects the block which adds them up -- lives in a file-scope __device__ array instead of the handle's workspace:
// no handle, no workspace, no cudaMalloc / cudaFree / allocating library call anywhere on this path.
//
// The array is per device (every GPU that loads libwl holds its 1 MiB + 256 B until the process exits) and shared by all calls:
// calls that overlap on the GPU (two streams, two host threads) RACE on it; calls on one stream are ordered and safe.  It keeps
// the previous call's contents: the counter is cleared on the stream before every launch, the partial sums are all rewritten
// before they are read (every block of a launch writes its own pair).
#include <cstdio>
#include <cstring>
#include <mutex>
#include <cuda_runtime.h>
#include "../../include/wl.h"

#define NS_NT 256                                        // threads per block
#define NS_CPB 1024                                      // cells per block (four per thread)
#define NS_MAXP (WL_STATIC_MAX_CELLS / NS_CPB)           // partial-sum pairs: one per block
#define NS_HEAD 256                                      // bytes in front of the partial sums: the ticket counter

// In HOST code this name is a host-side stand-in, not a device address: the address a kernel may use comes from
// cudaGetSymbolAddress (ns_scratch_ptr below), once per device.
static __device__ __align__(256) unsigned char wl_static_scratch[NS_HEAD + 16 * NS_MAXP];

__device__ __forceinline__ double ns_warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// u: ND component arrays of (n0+2)(n1+2)[(n2+2)] floats, x fastest, ghost layer included.  out[0] = 1/2 sum u_i^2,
// out[1] = 1/2 sum |w|^2 over the interior cells, w = the circulations around the cell edges through the lower corner of the
// cell (the differences k_energy takes).  fp32 products per cell, fp64 sums, fixed order: the same bits from run to run.
template <int ND>
__global__ void __launch_bounds__(NS_NT) k_energy_static(const float* __restrict__ u, int n0, int n1, int n2, long long ncells,
                                                         unsigned char* scratch, double* __restrict__ out)
{
    __shared__ double sm[2][NS_NT / 32];
    __shared__ bool is_last;
    unsigned* counter = reinterpret_cast<unsigned*>(scratch);
    double* part = reinterpret_cast<double*>(scratch + NS_HEAD);
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const long long S0 = n0 + 2, S01 = S0 * (n1 + 2), comp = S01 * (ND == 3 ? n2 + 2 : 1);
    const float* ux = u; const float* uy = u + comp; const float* uz = u + 2 * comp;
    double ke = 0.0, en = 0.0;
#pragma unroll
    for (int j = 0; j < NS_CPB / NS_NT; ++j) {
        const long long idx = (long long)blockIdx.x * NS_CPB + j * NS_NT + tid;
        if (idx >= ncells) continue;
        const int c0 = (int)(idx % n0);
        const long long t = idx / n0;
        const int c1 = (int)(t % n1), c2 = (int)(t / n1);
        const long long i = (c0 + 1) + S0 * (c1 + 1) + (ND == 3 ? S01 * (c2 + 1) : 0);
        const float a = __ldg(ux + i), b = __ldg(uy + i);
        const float wz = (b - __ldg(uy + i - 1)) - (a - __ldg(ux + i - S0));
        float k2 = a * a + b * b, w2 = wz * wz;
        if (ND == 3) {
            const float c = __ldg(uz + i);
            const float wx = (c - __ldg(uz + i - S0)) - (b - __ldg(uy + i - S01));
            const float wy = (a - __ldg(ux + i - S01)) - (c - __ldg(uz + i - 1));
            k2 += c * c;
            w2 += wx * wx + wy * wy;
        }
        ke += 0.5 * (double)k2;
        en += 0.5 * (double)w2;
    }
    // block sum -> this block's pair of partials
    ke = ns_warp_sum(ke); en = ns_warp_sum(en);
    if (lane == 0) { sm[0][wid] = ke; sm[1][wid] = en; }
    __syncthreads();
    if (tid == 0) {
        double a = 0.0, b = 0.0;
#pragma unroll
        for (int w = 0; w < NS_NT / 32; ++w) { a += sm[0][w]; b += sm[1][w]; }
        part[2 * (long long)blockIdx.x] = a;
        part[2 * (long long)blockIdx.x + 1] = b;
        __threadfence();
        const unsigned ticket = atomicAdd(counter, 1u);
        is_last = ticket == gridDim.x - 1;
    }
    __syncthreads();
    if (!is_last) return;
    // the last block to finish adds the partials of all blocks in a fixed order
    __threadfence();
    double a = 0.0, b = 0.0;
    for (long long k = tid; k < (long long)gridDim.x; k += NS_NT) { a += __ldcg(part + 2 * k); b += __ldcg(part + 2 * k + 1); }
    a = ns_warp_sum(a); b = ns_warp_sum(b);
    __syncthreads();
    if (lane == 0) { sm[0][wid] = a; sm[1][wid] = b; }
    __syncthreads();
    if (tid == 0) {
        double x = 0.0, y = 0.0;
#pragma unroll
        for (int w = 0; w < NS_NT / 32; ++w) { x += sm[0][w]; y += sm[1][w]; }
        out[0] = x;
        out[1] = y;
        *counter = 0u;
    }
}

// device address of the scratch array on the CURRENT device; looked up once per device (set-up), cached afterwards
#define NS_MAX_DEVICES 64
static std::mutex ns_mutex;
static void* ns_ptr[NS_MAX_DEVICES];

static cudaError_t ns_scratch_ptr(unsigned char** p)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= NS_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(ns_mutex);
    if (!ns_ptr[dev]) {
        void* q = nullptr;
        e = cudaGetSymbolAddress(&q, wl_static_scratch);
        if (e != cudaSuccess) return e;
        ns_ptr[dev] = q;
    }
    *p = static_cast<unsigned char*>(ns_ptr[dev]);
    return cudaSuccess;
}

static int ns_fail(int code, char* err, size_t err_len, const char* text)
{
    if (err && err_len) { strncpy(err, text, err_len - 1); err[err_len - 1] = 0; }
    return code;
}

extern "C" int wl_energy_static(const float* u_dev, int ndim, const int* dims, void* cuda_stream, double* out_dev, char* err, size_t err_len)
{
    char msg[256];
    if (err && err_len) err[0] = 0;
    if (!u_dev || !dims || !out_dev) return ns_fail(WL_EINVAL, err, err_len, "wl_energy_static: null pointer (u_dev, dims, out_dev are required)");
    if (ndim != 2 && ndim != 3) return ns_fail(WL_EINVAL, err, err_len, "wl_energy_static: ndim must be 2 or 3");
    long long ncells = 1;
    for (int d = 0; d < ndim; ++d) {
        if (dims[d] < 1 || dims[d] > (1 << 24)) return ns_fail(WL_EINVAL, err, err_len, "wl_energy_static: every dims[d] must lie in 1 .. 2^24");
        ncells *= dims[d];
        if (ncells > (long long)WL_STATIC_MAX_CELLS) {
            snprintf(msg, sizeof msg, "wl_energy_static: the grid exceeds the static scratch limit WL_STATIC_MAX_CELLS = %lld interior cells "
                                      "(one pair of partial sums per 1024 cells in a fixed 1 MiB device array); use wl_energy on a handle instead",
                     (long long)WL_STATIC_MAX_CELLS);
            return ns_fail(WL_ETOOBIG, err, err_len, msg);
        }
    }
    unsigned char* scratch = nullptr;
    cudaError_t e = ns_scratch_ptr(&scratch);
    if (e != cudaSuccess) {
        snprintf(msg, sizeof msg, "wl_energy_static: cudaGetSymbolAddress of the scratch array failed: %s", cudaGetErrorString(e));
        return ns_fail(WL_ECUDA, err, err_len, msg);
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const unsigned blocks = (unsigned)((ncells + NS_CPB - 1) / NS_CPB);
    // the array keeps whatever the last call (or an aborted one) left: the ticket counter must start at zero
    e = cudaMemsetAsync(scratch, 0, NS_HEAD, st);
    if (e == cudaSuccess) {
        if (ndim == 3) k_energy_static<3><<<blocks, NS_NT, 0, st>>>(u_dev, dims[0], dims[1], dims[2], ncells, scratch, out_dev);
        else           k_energy_static<2><<<blocks, NS_NT, 0, st>>>(u_dev, dims[0], dims[1], 1, ncells, scratch, out_dev);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        snprintf(msg, sizeof msg, "wl_energy_static: CUDA error: %s", cudaGetErrorString(e));
        return ns_fail(WL_ECUDA, err, err_len, msg);
    }
    return WL_OK;
}
