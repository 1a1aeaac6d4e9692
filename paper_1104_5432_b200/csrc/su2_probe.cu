// su2_probe.cu — memory-bandwidth probes behind su2_bandwidth_probe (include/su2_heatbath.h).
//
// the 32^4 fp32 lattice (64 MiB) lives in the 126 MB L2, so its
// roofline denominator is the L2 bandwidth of the box, which nobody publishes: measure it here, with
// the access shape of the path (128-bit loads, unit stride across a warp, every SM busy) and no
// arithmetic. The same kernels over a buffer larger than L2 give the HBM figure of the same run.
#include "su2_launch.h"

namespace su2 {

// grid-stride read of n uint4; the XOR keeps the loads alive, the store never happens in practice
__global__ void __launch_bounds__(256) probe_read_kernel(const uint4* __restrict__ src, size_t n, uint4* __restrict__ sink)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint4 acc = {0u, 0u, 0u, 0u};
    // 4 independent 128-bit loads in flight per thread and iteration
    for (; i + 3 * stride < n; i += 4 * stride) {
        uint4 a, b, c, d;
        asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w) : "l"(src + i));
        asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w) : "l"(src + i + stride));
        asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(c.x), "=r"(c.y), "=r"(c.z), "=r"(c.w) : "l"(src + i + 2 * stride));
        asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(d.x), "=r"(d.y), "=r"(d.z), "=r"(d.w) : "l"(src + i + 3 * stride));
        acc.x ^= a.x ^ b.x ^ c.x ^ d.x;
        acc.y ^= a.y ^ b.y ^ c.y ^ d.y;
        acc.z ^= a.z ^ b.z ^ c.z ^ d.z;
        acc.w ^= a.w ^ b.w ^ c.w ^ d.w;
    }
    for (; i < n; i += stride) {
        uint4 a;
        asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w) : "l"(src + i));
        acc.x ^= a.x; acc.y ^= a.y; acc.z ^= a.z; acc.w ^= a.w;
    }
    if ((acc.x & acc.y & acc.z & acc.w) == 0xFFFFFFFFu && sink) sink[0] = acc;  // buffer is zero-filled: never true
}

// grid-stride copy of n uint4 (read + write traffic: the shape of MEASURED_PEAKS.json's hbm_gbs)
__global__ void __launch_bounds__(256) probe_copy_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst, size_t n)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        uint4 a;
        asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w) : "l"(src + i));
        dst[i] = a;
    }
}

// Runs `passes` launches over `bytes` of a zero-filled device buffer (two untimed ones first, which also
// make a buffer that fits L2 resident) and returns GB/s of algorithmic traffic: bytes per pass for a read,
// 2 x bytes/2 = bytes for a copy of the first half onto the second. CUDA events on the launching stream.
int run_bandwidth_probe(size_t bytes, int passes, int mode, cudaStream_t st, double* gbs_out, double* us_per_pass_out)
{
    void* buf = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t ce = cudaMalloc(&buf, bytes);
    if (ce == cudaSuccess) ce = cudaMemsetAsync(buf, 0, bytes, st);
    if (ce == cudaSuccess) ce = cudaEventCreate(&e0);
    if (ce == cudaSuccess) ce = cudaEventCreate(&e1);
    int dev = 0, sms = 148;
    if (ce == cudaSuccess) ce = cudaGetDevice(&dev);
    if (ce == cudaSuccess) ce = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const unsigned grid = (unsigned)sms * 8u;  // 8 CTAs of 256 threads per SM: every SM full
    const size_t n = bytes / sizeof(uint4);
    float ms = 0.f;
    if (ce == cudaSuccess) {
        for (int i = -2; i < passes; ++i) {
            if (i == 0) cudaEventRecord(e0, st);
            if (mode == 0)
                probe_read_kernel<<<grid, 256, 0, st>>>((const uint4*)buf, n, nullptr);
            else
                probe_copy_kernel<<<grid, 256, 0, st>>>((const uint4*)buf, (uint4*)buf + n / 2, n / 2);
        }
        cudaEventRecord(e1, st);
        ce = cudaEventSynchronize(e1);
        if (ce == cudaSuccess) ce = cudaGetLastError();
        if (ce == cudaSuccess) ce = cudaEventElapsedTime(&ms, e0, e1);
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (buf) cudaFree(buf);
    if (ce != cudaSuccess) {
        cudaGetLastError();
        return (ce == cudaErrorMemoryAllocation) ? 2 : 3;
    }
    const double sec = (double)ms * 1e-3 / passes;
    *gbs_out = (double)(n * sizeof(uint4)) / sec / 1e9;
    if (us_per_pass_out) *us_per_pass_out = sec * 1e6;
    return 0;
}

}  // namespace su2
