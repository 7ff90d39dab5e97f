// hough_microbench.cu -- shared-memory atomic micro-benchmark that DEFINES the
// "shared-atomic roofline" the vote kernel is reported against (SURVEY.md section 8(d),
// BASELINE.json north_star "% of smem-atomic roofline").  Not part of the hot path.
#include <atomic>

#include "hough_internal.cuh"

#define MB_WORDS 8192 // 32 KB table per CTA

template <int MODE>
__global__ void __launch_bounds__(1024) k_microbench(int iters, uint32_t *sink)
{
    __shared__ uint32_t table[MB_WORDS];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int w = tid; w < MB_WORDS; w += blockDim.x)
        table[w] = 0u;
    __syncthreads();
    const uint32_t bit = 1u << (tid & 15);
    uint32_t rnd = tid * 2654435761u + 12345u;
    uint32_t base = (uint32_t)(warp * 64 + lane);
#pragma unroll 8
    for (int it = 0; it < iters; ++it) {
        uint32_t idx;
        if (MODE == 1) {
            rnd = rnd * 1664525u + 1013904223u;
            idx = (rnd >> 9) & (MB_WORDS - 1);
        } else {
            idx = (base + (uint32_t)it * 32u) & (MB_WORDS - 1); // 32 lanes -> 32 distinct banks
        }
        if (MODE == 2) {
            volatile uint32_t *t = table;
            t[idx] = t[idx] | bit;
        } else {
            atomicOr(&table[idx], bit);
        }
    }
    __syncthreads();
    uint32_t acc = 0u;
    for (int w = tid; w < MB_WORDS; w += blockDim.x)
        acc ^= table[w];
    if (acc == 0xdeadbeefu)
        sink[0] = acc;
}

int hough_microbench_smem(int device, int mode, int threads, int ctas_per_sm, int iters, uint32_t *sink_dev,
                          void *cuda_stream, uint64_t *lane_ops)
{
    if (mode < 0 || mode > 2 || threads < 32 || threads > 1024 || (threads & 31) || ctas_per_sm < 1 ||
        iters < 1 || !sink_dev)
        return HOUGH_EINVAL;
    // The caller times this call with events recorded around it, so after the first call on a device nothing
    // but the launch may sit between them: the SM count is looked up once per device and remembered.
    static std::atomic<int> sm_count[64];
    if (device < 0 || device >= 64)
        return HOUGH_ECUDA;
    int sms = sm_count[device].load(std::memory_order_relaxed);
    if (sms == 0) {
        int ndev = 0;
        if (cudaGetDeviceCount(&ndev) != cudaSuccess || device >= ndev) {
            cudaGetLastError();
            return HOUGH_ECUDA;
        }
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || sms < 1) {
            cudaGetLastError();
            return HOUGH_ECUDA;
        }
        sm_count[device].store(sms, std::memory_order_relaxed);
    }
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || (cur != device && cudaSetDevice(device) != cudaSuccess)) {
        cudaGetLastError();
        return HOUGH_ECUDA;
    }
    int blocks = sms * ctas_per_sm;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (mode == 0)
        k_microbench<0><<<blocks, threads, 0, st>>>(iters, sink_dev);
    else if (mode == 1)
        k_microbench<1><<<blocks, threads, 0, st>>>(iters, sink_dev);
    else
        k_microbench<2><<<blocks, threads, 0, st>>>(iters, sink_dev);
    if (cudaGetLastError() != cudaSuccess)
        return HOUGH_ECUDA;
    if (lane_ops)
        *lane_ops = (uint64_t)blocks * (uint64_t)threads * (uint64_t)iters;
    return HOUGH_OK;
}
