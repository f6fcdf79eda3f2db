// oat_penalty_value_noalloc (include/oat.h): the smoothness penalty R(x) = x^T L x of Eq. (34) L305 (reading G21) for
// callers that must not allocate device memory.
//
// Who that is: code that runs after the application has handed every free byte of the GPU to its own pool (a cudaMalloc
// then fails, or succeeds only by shrinking the pool), and real-time acquisition loops in which a cudaMalloc / cudaFree
// is not acceptable because both synchronise the whole device and stall every other stream.  oat_penalty_value is
// closed to them twice over: it needs a geometry handle (whose creation allocates its tables) and it sizes a
// volume-long scratch buffer with cudaMalloc on first use.
//
// This file is the same computation -- the stencil pass that writes L x to scratch, then the fp64 dot product <x, L x>
// -- with the scratch in the library's own image: one file-scope __device__ array, fixed at build time, present on
// every GPU that loads liboat.so for as long as the process lives.  Nothing here calls cudaMalloc, cudaFree,
// cudaMallocHost or a library routine that allocates.
//
// The arithmetic, the launch shapes and the summation widths are those of oat_penalty_kernel (oat_next.cu) and
// oat_dot_kernel (oat_kernels.cu); the existing entry points and kernels are untouched.
#include "../../include/oat.h"
#include "oat_internal.h"

#include <mutex>

namespace {

// Scratch layout: [0, 256) header, of which the first 8 bytes are the fp64 accumulator of the dot product;
// [256, 256 + 4 * OAT_NOALLOC_MAX_VOXELS) the fp32 volume L x.  8 MiB + 256 B per GPU.
constexpr size_t kHeaderBytes = 256;
constexpr size_t kScratchBytes = kHeaderBytes + sizeof(float) * (size_t)OAT_NOALLOC_MAX_VOXELS;

// In HOST code this name is only a stand-in for the symbol (its host address is not device memory): the device
// address is asked for once per device with cudaGetSymbolAddress below and only that pointer is handed to kernels.
static __device__ __align__(256) unsigned char oat_noalloc_scratch[kScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_setup_lock;
void *g_scratch_of_device[kMaxDevices] = {};     // device address of the array on each ordinal, nullptr = not set up yet

// Once per device, with that device current: resolve the array's address there.  No allocation: the array already
// exists on the device as part of the loaded module (the lookup makes the runtime load the module if this is the first
// use of liboat.so on that device, which is why the first call belongs outside a stream capture).
int scratch_on_current_device(int dev, unsigned char **out)
{
    std::lock_guard<std::mutex> hold(g_setup_lock);
    if (!g_scratch_of_device[dev]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, oat_noalloc_scratch);
        if (e != cudaSuccess || !p)
            return oat_fail(OAT_ERR_CUDA, "cudaGetSymbolAddress(oat_noalloc_scratch) failed on device %d: %s", dev,
                            cudaGetErrorString(e));
        g_scratch_of_device[dev] = p;
    }
    *out = static_cast<unsigned char *>(g_scratch_of_device[dev]);
    return OAT_OK;
}

// Same sizing rule as the other vector kernels of the library (a few waves over the 148 SMs, grid-stride beyond).
inline int grid_for(long long n, int block)
{
    long long g = (n + block - 1) / block;
    const long long cap = 148LL * 16;
    if (g > cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

// lx[n] = (L x)_n: per axis (x_n - x_before) + (x_n - x_after), a term only where that neighbour exists (Eq. 34,
// reading G21).  Every element of lx[0, n) is written, so nothing of the previous call's L x survives into this one.
__global__ void oat_penalty_noalloc_kernel(int nx, int ny, int nz, const float *__restrict__ x, float *__restrict__ lx)
{
    const long long n = (long long)nx * ny * nz;
    const long long sy = nx, sz = (long long)nx * ny;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int ix = (int)(i % nx);
        const long long r = i / nx;
        const int iy = (int)(r % ny), iz = (int)(r / ny);
        const float c = x[i];
        float s = 0.f;
        if (ix > 0) s += c - x[i - 1];
        if (ix + 1 < nx) s += c - x[i + 1];
        if (iy > 0) s += c - x[i - sy];
        if (iy + 1 < ny) s += c - x[i + sy];
        if (iz > 0) s += c - x[i - sz];
        if (iz + 1 < nz) s += c - x[i + sz];
        lx[i] = s;
    }
}

__device__ __forceinline__ double warp_sum(double v)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// *acc += <a, b> in fp64; *acc is the header word of the scratch array and was zeroed on the stream before this launch.
__global__ void oat_dot_noalloc_kernel(const float *__restrict__ a, const float *__restrict__ b, long long n, double *acc)
{
    double s = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        s += (double)a[i] * (double)b[i];
    s = warp_sum(s);
    __shared__ double sh[32];
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        double v = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
        v = warp_sum(v);
        if (threadIdx.x == 0) atomicAdd(acc, v);
    }
}

#define NOALLOC_TRY(expr)                                                                                         \
    do {                                                                                                          \
        cudaError_t e_ = (expr);                                                                                  \
        if (e_ != cudaSuccess) return oat_fail(OAT_ERR_CUDA, "%s failed: %s", #expr, cudaGetErrorString(e_));     \
    } while (0)

}  // namespace

int oat_penalty_value_noalloc(int32_t nx, int32_t ny, int32_t nz, const float *d_x, double *h_value, void *cuda_stream)
{
    if (nx < 1 || ny < 1 || nz < 1) return oat_fail(OAT_ERR_INVALID, "nx, ny, nz must be >= 1 (got %d, %d, %d)", nx, ny, nz);
    if (!d_x || !h_value) return oat_fail(OAT_ERR_INVALID, "d_x / h_value must not be NULL");
    const long long n = (long long)nx * ny * nz;
    if (n > (long long)OAT_NOALLOC_MAX_VOXELS)
        return oat_fail(OAT_ERR_INVALID,
                        "oat_penalty_value_noalloc: %d x %d x %d = %lld voxels exceed the built-in scratch of %d voxels "
                        "(OAT_NOALLOC_MAX_VOXELS); use oat_penalty_value, which allocates its scratch, for larger volumes",
                        nx, ny, nz, n, (int)OAT_NOALLOC_MAX_VOXELS);
    int dev = -1;
    NOALLOC_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return oat_fail(OAT_ERR_INVALID, "device ordinal %d outside [0, %d)", dev, kMaxDevices);
    // a pointer query, not an allocation: refuse host memory and memory of another GPU before a kernel faults on it
    cudaPointerAttributes attr;
    NOALLOC_TRY(cudaPointerGetAttributes(&attr, d_x));
    if (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged)
        return oat_fail(OAT_ERR_INVALID, "d_x is not device memory");
    if (attr.type == cudaMemoryTypeDevice && attr.device != dev)
        return oat_fail(OAT_ERR_INVALID, "d_x lives on device %d but the calling thread's current device is %d", attr.device, dev);

    unsigned char *scratch = nullptr;
    int rc = scratch_on_current_device(dev, &scratch);
    if (rc) return rc;
    double *acc = reinterpret_cast<double *>(scratch);
    float *lx = reinterpret_cast<float *>(scratch + kHeaderBytes);

    cudaStream_t st = (cudaStream_t)cuda_stream;
    NOALLOC_TRY(cudaMemsetAsync(acc, 0, sizeof(double), st));      // the array keeps the last call's sum: start from zero
    oat_penalty_noalloc_kernel<<<grid_for(n, 256), 256, 0, st>>>(nx, ny, nz, d_x, lx);
    oat_dot_noalloc_kernel<<<grid_for(n, 256), 256, 0, st>>>(d_x, lx, n, acc);
    NOALLOC_TRY(cudaGetLastError());
    NOALLOC_TRY(cudaMemcpyAsync(h_value, acc, sizeof(double), cudaMemcpyDeviceToHost, st));
    NOALLOC_TRY(cudaStreamSynchronize(st));
    return OAT_OK;
}
