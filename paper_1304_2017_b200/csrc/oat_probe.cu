// Measurement aids of liboat.so (include/oat_probe.h): micro-benchmarks of the two hardware paths the marching kernels
// lean on -- scattered 256-bit loads that miss L1 (H) and 16-byte vector reductions into L2 (H^T).  They are NOT part of
// the product ABI and nothing on the operator path calls them; bench.py reports their figures as diagnostics only.
#include "../../include/oat_probe.h"
#include "oat_internal.h"

#include <stdarg.h>
#include <stdio.h>

namespace {

__device__ __forceinline__ void red_add_v4(float4 *addr, float a, float b, float c, float d)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

// probe for oat_measure_red_rate(): every lane adds a float4 into its own pseudo-random 32-byte sector
__global__ void oat_red_probe_kernel(float4 *__restrict__ buf, unsigned n16, int iters)
{
    const unsigned lane = threadIdx.x & 31, gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    unsigned s = gw * 2654435761u + 12345u;
    for (int i = 0; i < iters; ++i) {
        s = s * 1664525u + 1013904223u;
        const unsigned h = (s >> 4) + lane * 2654435761u;
        const unsigned r = ((h ^ (h >> 13)) * 0x9E3779B1u) % (n16 / 2);
        red_add_v4(buf + 2 * (size_t)r, 1.f, 1.f, 1.f, 1.f);
    }
}

// probe for oat_measure_gather_rate(): every lane loads its own pseudo-random 32-byte sector (one 256-bit load, the
// access of consume_march_fwd), four independent loads in flight per thread; the sum keeps the loads alive
__global__ void oat_gather_probe_kernel(const float4 *__restrict__ buf, unsigned n16, int iters, float *__restrict__ sink)
{
    const unsigned lane = threadIdx.x & 31, gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    unsigned s = gw * 2654435761u + 54321u;
    float acc = 0.f;
    for (int i = 0; i < iters; ++i) {
        float v[4][8];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            s = s * 1664525u + 1013904223u;
            const unsigned h = (s >> 4) + lane * 2654435761u;
            const unsigned r = ((h ^ (h >> 13)) * 0x9E3779B1u) % (n16 / 2);
            asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                         : "=f"(v[u][0]), "=f"(v[u][1]), "=f"(v[u][2]), "=f"(v[u][3]), "=f"(v[u][4]), "=f"(v[u][5]), "=f"(v[u][6]), "=f"(v[u][7])
                         : "l"(buf + 2 * (size_t)r));
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) acc += v[u][0] + v[u][7];
    }
    if (acc == 12345.678f) sink[0] = acc;
}

// probe for oat_measure_gather_rate_ex(): `active` of the 32 lanes load one pseudo-random sector each, ONE load in flight
// per thread (its result is consumed before the next is issued) -- the request shape of the marching loop of H;
// dynamic shared memory (unused) sets the shared-memory carve-out and with it the size of L1
__global__ void __launch_bounds__(128, 8) oat_gather_probe_ex_kernel(const float4 *__restrict__ buf, unsigned nsec, int iters, int active, float *__restrict__ sink)
{
    const unsigned lane = threadIdx.x & 31, gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    unsigned s = gw * 2654435761u + 54321u;
    float acc = 0.f;
    const bool act = (int)((lane * 7) & 31) < active;
    for (int i = 0; i < iters; ++i) {
        float v[8];
        s = s * 1664525u + 1013904223u;
        const unsigned h = (s >> 4) + lane * 2654435761u;
        const unsigned r = ((h ^ (h >> 13)) * 0x9E3779B1u) & (nsec - 1);      // nsec is a power of two
        if (act) {
            asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                         : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7])
                         : "l"(buf + 2 * (size_t)r));
            acc += v[0] + v[7];
        }
    }
    if (acc == 12345.678f) sink[0] = acc;
}

// probe for oat_measure_red_rate_ex(): RED.128 with a chosen address pattern within the warp
__global__ void oat_red_probe_ex_kernel(float4 *__restrict__ buf, unsigned n16, int iters, int pattern)
{
    const unsigned lane = threadIdx.x & 31, gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    unsigned s = gw * 2654435761u + 12345u;
    for (int i = 0; i < iters; ++i) {
        s = s * 1664525u + 1013904223u;
        const unsigned wbase = ((s >> 4) ^ (s >> 17)) * 0x9E3779B1u;       // the same for all lanes of the warp
        unsigned r;
        if (pattern == 0) { const unsigned h = (s >> 4) + lane * 2654435761u; r = (h ^ (h >> 13)) * 0x9E3779B1u; }   // every lane its own record
        else if (pattern == 1) r = wbase + lane;                           // 32 consecutive records = 16 sectors in 4 lines
        else if (pattern == 2) r = wbase + lane * 8;                       // one record per 128-byte line, 32 lines
        else if (pattern == 3) r = wbase + (lane >> 1) * 64 + (lane & 1);  // lane pairs share a sector, pairs 1 KB apart
        else if (pattern == 4) r = wbase + (lane >> 3) * 1024 + (lane & 7);  // 4 scattered lines of 8 records
        else if (pattern == 5) { const unsigned h = (s >> 4) + lane * 2654435761u; r = ((h ^ (h >> 13)) * 0x9E3779B1u) & ~1u; }   // own sector, both halves (below)
        else if (pattern == 6) { const unsigned h = (s >> 4) + (lane & 15) * 2654435761u; r = (((h ^ (h >> 13)) * 0x9E3779B1u) & ~1u) + (lane >> 4); }   // lanes l, l + 16 fill one scattered sector
        else { const unsigned h = (s >> 4) + (lane >> 1) * 2654435761u; r = (((h ^ (h >> 13)) * 0x9E3779B1u) & ~1u) + (lane & 1); }      // lanes 2m, 2m + 1 fill one scattered sector
        if (pattern == 5) {
            // the face-quad case "flush L and H of one cell": one thread, two back-to-back reductions into the two
            // 16-byte halves of ONE scattered 32-byte sector (n16 is even, so r + 1 stays inside the buffer)
            float4 *p = buf + (r % n16);
            red_add_v4(p, 1.f, 1.f, 1.f, 1.f);
            red_add_v4(p + 1, 1.f, 1.f, 1.f, 1.f);
        } else
            red_add_v4(buf + (r % n16), 1.f, 1.f, 1.f, 1.f);
    }
}

}  // namespace

static void oat_launch_red_probe(float4 *buf, unsigned n16, int iters, int blocks, cudaStream_t st)
{
    oat_red_probe_kernel<<<blocks, 256, 0, st>>>(buf, n16, iters);
}

static void oat_launch_gather_probe(const float4 *buf, unsigned n16, int iters, int blocks, float *sink, cudaStream_t st)
{
    oat_gather_probe_kernel<<<blocks, 256, 0, st>>>(buf, n16, iters, sink);
}

static cudaError_t oat_launch_gather_probe_ex(const float4 *buf, unsigned nsec, int iters, int active, int smem_bytes, int blocks, float *sink, cudaStream_t st)
{
    cudaError_t e = cudaFuncSetAttribute(oat_gather_probe_ex_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
    if (e != cudaSuccess) return e;
    oat_gather_probe_ex_kernel<<<blocks, 128, smem_bytes, st>>>(buf, nsec, iters, active, sink);
    return cudaGetLastError();
}

static void oat_launch_red_probe_ex(float4 *buf, unsigned n16, int iters, int pattern, int blocks, cudaStream_t st)
{
    oat_red_probe_ex_kernel<<<blocks, 256, 0, st>>>(buf, n16, iters, pattern);
}

#define CUDA_TRY(expr)                                                                          \
    do {                                                                                        \
        cudaError_t e_ = (expr);                                                                \
        if (e_ != cudaSuccess)                                                                  \
            return oat_fail(e_ == cudaErrorMemoryAllocation ? OAT_ERR_ALLOC : OAT_ERR_CUDA,     \
                            "%s failed: %s", #expr, cudaGetErrorString(e_));                    \
    } while (0)
#define fail oat_fail

extern "C" {

int oat_measure_red_rate(int device, double *lanes_per_s)
{
    if (!lanes_per_s) return fail(OAT_ERR_INVALID, "NULL argument");
    CUDA_TRY(cudaSetDevice(device));
    const size_t bytes = 64u << 20;                       // L2-resident
    const int blocks = 148 * 8, iters = 2000;
    float4 *buf = nullptr;
    cudaEvent_t a = nullptr, b = nullptr;
    CUDA_TRY(cudaMalloc((void **)&buf, bytes));
    cudaError_t e = cudaMemset(buf, 0, bytes);
    if (e == cudaSuccess) e = cudaEventCreate(&a);
    if (e == cudaSuccess) e = cudaEventCreate(&b);
    float ms = 0.f;
    if (e == cudaSuccess) {
        oat_launch_red_probe(buf, (unsigned)(bytes / 16), 200, blocks, 0);      // warm-up
        cudaEventRecord(a, 0);
        oat_launch_red_probe(buf, (unsigned)(bytes / 16), iters, blocks, 0);
        cudaEventRecord(b, 0);
        e = cudaEventSynchronize(b);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
    }
    if (a) cudaEventDestroy(a);
    if (b) cudaEventDestroy(b);
    cudaFree(buf);
    if (e != cudaSuccess || !(ms > 0.f)) return fail(OAT_ERR_CUDA, "reduction-rate probe failed: %s", cudaGetErrorString(e));
    *lanes_per_s = (double)blocks * 256.0 * iters / (ms * 1e-3);
    return OAT_OK;
}

int oat_measure_gather_rate(int device, double *sectors_per_s)
{
    if (!sectors_per_s) return fail(OAT_ERR_INVALID, "NULL argument");
    CUDA_TRY(cudaSetDevice(device));
    const size_t bytes = 64u << 20;                       // L2-resident, far larger than L1
    const int blocks = 148 * 8, iters = 500;
    float4 *buf = nullptr;
    float *sink = nullptr;
    cudaEvent_t a = nullptr, b = nullptr;
    CUDA_TRY(cudaMalloc((void **)&buf, bytes));
    cudaError_t e = cudaMemset(buf, 0, bytes);
    if (e == cudaSuccess) e = cudaMalloc((void **)&sink, sizeof(float));
    if (e == cudaSuccess) e = cudaEventCreate(&a);
    if (e == cudaSuccess) e = cudaEventCreate(&b);
    float ms = 0.f;
    if (e == cudaSuccess) {
        oat_launch_gather_probe(buf, (unsigned)(bytes / 16), 50, blocks, sink, 0);      // warm-up (fills L2)
        cudaEventRecord(a, 0);
        oat_launch_gather_probe(buf, (unsigned)(bytes / 16), iters, blocks, sink, 0);
        cudaEventRecord(b, 0);
        e = cudaEventSynchronize(b);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
    }
    if (a) cudaEventDestroy(a);
    if (b) cudaEventDestroy(b);
    cudaFree(sink);
    cudaFree(buf);
    if (e != cudaSuccess || !(ms > 0.f)) return fail(OAT_ERR_CUDA, "gather-rate probe failed: %s", cudaGetErrorString(e));
    *sectors_per_s = (double)blocks * 256.0 * 4.0 * iters / (ms * 1e-3);
    return OAT_OK;
}

int oat_measure_gather_rate_ex(int device, int lanes_active, int smem_kb_per_block, double *sectors_per_s)
{
    if (!sectors_per_s || lanes_active < 1 || lanes_active > 32 || smem_kb_per_block < 0 || smem_kb_per_block > 27)
        return fail(OAT_ERR_INVALID, "bad argument (lanes_active 1..32, smem_kb_per_block 0..27)");
    CUDA_TRY(cudaSetDevice(device));
    const size_t bytes = 64u << 20;
    const int blocks = 148 * 8, iters = 2000;
    float4 *buf = nullptr; float *sink = nullptr;
    cudaEvent_t a = nullptr, b = nullptr;
    CUDA_TRY(cudaMalloc((void **)&buf, bytes));
    cudaError_t e = cudaMemset(buf, 0, bytes);
    if (e == cudaSuccess) e = cudaMalloc((void **)&sink, sizeof(float));
    if (e == cudaSuccess) e = cudaEventCreate(&a);
    if (e == cudaSuccess) e = cudaEventCreate(&b);
    float ms = 0.f;
    if (e == cudaSuccess) e = oat_launch_gather_probe_ex(buf, (unsigned)(bytes / 32), 100, lanes_active, smem_kb_per_block * 1024, blocks, sink, 0);
    if (e == cudaSuccess) {
        cudaEventRecord(a, 0);
        e = oat_launch_gather_probe_ex(buf, (unsigned)(bytes / 32), iters, lanes_active, smem_kb_per_block * 1024, blocks, sink, 0);
        cudaEventRecord(b, 0);
        if (e == cudaSuccess) e = cudaEventSynchronize(b);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
    }
    if (a) cudaEventDestroy(a);
    if (b) cudaEventDestroy(b);
    cudaFree(sink); cudaFree(buf);
    if (e != cudaSuccess || !(ms > 0.f)) return fail(OAT_ERR_CUDA, "gather-rate probe failed: %s", cudaGetErrorString(e));
    *sectors_per_s = (double)blocks * 4.0 * iters * lanes_active / (ms * 1e-3);
    return OAT_OK;
}

int oat_measure_red_rate_ex(int device, int pattern, double *lanes_per_s)
{
    if (!lanes_per_s || pattern < 0 || pattern > 7) return fail(OAT_ERR_INVALID, "bad argument (pattern 0..7)");
    CUDA_TRY(cudaSetDevice(device));
    const size_t bytes = 64u << 20;
    const int blocks = 148 * 8, iters = 2000;
    float4 *buf = nullptr;
    cudaEvent_t a = nullptr, b = nullptr;
    CUDA_TRY(cudaMalloc((void **)&buf, bytes));
    cudaError_t e = cudaMemset(buf, 0, bytes);
    if (e == cudaSuccess) e = cudaEventCreate(&a);
    if (e == cudaSuccess) e = cudaEventCreate(&b);
    float ms = 0.f;
    if (e == cudaSuccess) {
        oat_launch_red_probe_ex(buf, (unsigned)(bytes / 16), 200, pattern, blocks, 0);
        cudaEventRecord(a, 0);
        oat_launch_red_probe_ex(buf, (unsigned)(bytes / 16), iters, pattern, blocks, 0);
        cudaEventRecord(b, 0);
        e = cudaEventSynchronize(b);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
    }
    if (a) cudaEventDestroy(a);
    if (b) cudaEventDestroy(b);
    cudaFree(buf);
    if (e != cudaSuccess || !(ms > 0.f)) return fail(OAT_ERR_CUDA, "reduction-rate probe failed: %s", cudaGetErrorString(e));
    *lanes_per_s = (double)blocks * 256.0 * iters * (pattern == 5 ? 2.0 : 1.0) / (ms * 1e-3);    // pattern 5 issues two reductions per step
    return OAT_OK;
}


}  // extern "C"
