// hough_noalloc.cu -- hough_peaks_noalloc: peaks of a caller-supplied accumulator, with NO device
// allocation anywhere on the path (see include/hough.h for the contract).
//
// Who this is for.  Every other entry point of the library needs a handle, and a handle needs a
// workspace that somebody obtained from cudaMalloc (or torch).  Some users of a trigger library
// cannot do that: a plug-in that runs inside a host framework which owns the whole device-memory
// budget and only lends the plug-in its input and output buffers; a real-time event loop in which
// cudaMalloc / cudaFree are banned because they synchronise the whole device and so stall the events
// in flight on the other streams; a thin C or Fortran client that was handed device pointers by
// someone else and links no allocator of its own.  Such a caller still owns inputs and outputs.
// What it cannot provide is the SCRATCH the chained scan needs (its ticket and look-back words).
// Here that scratch is a file-scope __device__ array: it is part of the loaded module, so it exists
// on every GPU that loads libhough_b200.so from the moment the module is loaded until the process
// exits (65 792 bytes per GPU), and nobody has to allocate or free it.
//
// The kernel is a one-launch variant of the chained scan k_scan<SCAN_ROWS> (hough_peaks.cu): the
// same ticket order and decoupled look-back over 64-bit status words, but the items are the bins
// themselves, the peak test (rule A6 of DESIGN.md section 2, written out neighbour by neighbour)
// runs in front of the scan and the ordered compaction behind it.  It is the simple path, not the
// fast one: the streaming sweep + scan + compaction of hough_peaks stays the product hot path.
//
// Shares nothing with oracle/.
#include <mutex>

#include "hough_internal.cuh"

#define NA_THREADS 256
#define NA_PER_THREAD 8
#define NA_ITEMS (NA_THREADS * NA_PER_THREAD) // bins per block
#define NA_MAX_BLOCKS ((HOUGH_NOALLOC_MAX_BINS + NA_ITEMS - 1) / NA_ITEMS)
#define NA_HEAD_BYTES 256 // the ticket lives alone in the first 256 bytes
#define NA_SCRATCH_BYTES (NA_HEAD_BYTES + 8 * NA_MAX_BLOCKS)
#define NA_MAX_DEVICES 64

// The scratch of every call on this GPU.  In HOST code this name is only a stand-in for the
// symbol -- it is not a device address and must never be handed to a kernel or to cudaMemset;
// scratch_address() below asks the runtime for the real address once per device.
static __device__ __align__(256) unsigned char g_noalloc_scratch[NA_SCRATCH_BYTES];

struct NoallocParams {
    const uint32_t *acc;
    uint32_t n_bins;
    int n_phi, n_d0, n_kappa, L_min, wrap;
    uint32_t *bin, *mask, *n_peaks;
    uint32_t cap_peaks;
    unsigned int *ticket;       // scratch + 0
    unsigned long long *status; // scratch + NA_HEAD_BYTES, one word per block
};

// A6: pc >= L_min and the bin beats every existing neighbour, ties to the lower linear index.
__device__ __forceinline__ bool noalloc_is_peak(const NoallocParams &p, uint32_t lin)
{
    const int pc = __popc(p.acc[lin]);
    if (pc < p.L_min)
        return false;
    const int k = (int)(lin % (uint32_t)p.n_kappa);
    const uint32_t row = lin / (uint32_t)p.n_kappa;
    const int j = (int)(row % (uint32_t)p.n_d0), i = (int)(row / (uint32_t)p.n_d0);
    for (int di = -1; di <= 1; ++di) {
        int ii = i + di;
        if (ii < 0 || ii >= p.n_phi) {
            if (!p.wrap)
                continue;
            ii = ii < 0 ? ii + p.n_phi : ii - p.n_phi; // n_phi >= 3: three distinct rows
        }
        for (int dj = -1; dj <= 1; ++dj) {
            const int jj = j + dj;
            if (jj < 0 || jj >= p.n_d0)
                continue;
            for (int dk = -1; dk <= 1; ++dk) {
                const int kk = k + dk;
                if (kk < 0 || kk >= p.n_kappa || (di == 0 && dj == 0 && dk == 0))
                    continue;
                const uint32_t nl = ((uint32_t)ii * (uint32_t)p.n_d0 + (uint32_t)jj) * (uint32_t)p.n_kappa + (uint32_t)kk;
                const int pn = __popc(p.acc[nl]);
                if (pn > pc || (pn == pc && nl < lin))
                    return false;
            }
        }
    }
    return true;
}

__global__ void __launch_bounds__(NA_THREADS) k_peaks_noalloc(const NoallocParams p)
{
    __shared__ unsigned int s_ticket;
    __shared__ unsigned int s_warp[NA_THREADS / 32];
    __shared__ unsigned int s_prefix;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0)
        s_ticket = atomicAdd(p.ticket, 1u); // ticket order: a block only ever waits for blocks that already run
    __syncthreads();
    const unsigned int t = s_ticket;
    const uint32_t first = t * (uint32_t)NA_ITEMS + (uint32_t)tid * NA_PER_THREAD;

    uint32_t fl = 0;
#pragma unroll
    for (int q = 0; q < NA_PER_THREAD; ++q)
        if (first + q < p.n_bins && noalloc_is_peak(p, first + q))
            fl |= 1u << q;
    const unsigned int mine = __popc(fl);

    // exclusive scan of `mine` over the block
    unsigned int incl = mine;
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o)
            incl += y;
    }
    if (lane == 31)
        s_warp[warp] = incl;
    __syncthreads();
    unsigned int wbase = 0, agg = 0;
    for (int w = 0; w < NA_THREADS / 32; ++w) {
        const unsigned int x = s_warp[w];
        if (w < warp)
            wbase += x;
        agg += x;
    }
    const unsigned int texcl = wbase + incl - mine;

    // decoupled look-back: status word = (flag << 62) | value, flag 1 = this block's own sum,
    // 2 = sum of this block and everything before it; one 64-bit store carries both
    if (tid == 0) {
        volatile unsigned long long *status = p.status;
        const unsigned long long VAL = (1ull << 62) - 1ull;
        unsigned long long prefix = 0;
        if (t == 0) {
            status[0] = (2ull << 62) | agg;
        } else {
            status[t] = (1ull << 62) | agg;
            for (long long q = (long long)t - 1; q >= 0; --q) {
                unsigned long long sw;
                do {
                    sw = status[q];
                } while ((sw >> 62) == 0ull);
                prefix += sw & VAL;
                if ((sw >> 62) == 2ull)
                    break;
            }
            status[t] = (2ull << 62) | (prefix + agg);
        }
        s_prefix = (unsigned int)prefix;
    }
    __syncthreads();

    unsigned int rank = s_prefix + texcl;
#pragma unroll
    for (int q = 0; q < NA_PER_THREAD; ++q)
        if (fl & (1u << q)) {
            if (rank < p.cap_peaks) {
                p.bin[rank] = first + q;
                p.mask[rank] = p.acc[first + q];
            }
            ++rank;
        }
    // the block that holds the last bin knows the total
    if (tid == NA_THREADS - 1 && (unsigned long long)(t + 1u) * NA_ITEMS >= p.n_bins)
        *p.n_peaks = rank;
}

// Device address of g_noalloc_scratch on the CURRENT device, asked for once per device.
static int scratch_address(unsigned char **out)
{
    static std::mutex mu;
    static unsigned char *addr[NA_MAX_DEVICES];
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= NA_MAX_DEVICES)
        return HOUGH_ECUDA;
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        unsigned char *ptr = nullptr;
        if (cudaGetSymbolAddress((void **)&ptr, g_noalloc_scratch) != cudaSuccess || !ptr) {
            (void)cudaGetLastError();
            return HOUGH_ECUDA;
        }
        addr[dev] = ptr;
    }
    *out = addr[dev];
    return HOUGH_OK;
}

extern "C" int hough_peaks_noalloc(const uint32_t *acc, int32_t n_phi, int32_t n_d0, int32_t n_kappa, int32_t L_min,
                                   int32_t phi_wrap, uint32_t *bin, uint32_t *mask, uint32_t cap_peaks,
                                   uint32_t *n_peaks, void *cuda_stream)
{
    if (!acc || !bin || !mask || !n_peaks || cap_peaks == 0u)
        return HOUGH_EINVAL;
    if (n_phi < 1 || n_d0 < 1 || n_kappa < 1 || L_min < 1 || L_min > 32)
        return HOUGH_EINVAL;
    if ((phi_wrap != 0 && phi_wrap != 1) || (phi_wrap && n_phi < 3))
        return HOUGH_EINVAL;
    const unsigned long long n_bins = (unsigned long long)n_phi * (unsigned long long)n_d0 * (unsigned long long)n_kappa;
    if (n_bins > (unsigned long long)HOUGH_NOALLOC_MAX_BINS)
        return HOUGH_ENOMEM; // the fixed scratch holds look-back words for HOUGH_NOALLOC_MAX_BINS bins, no more
    unsigned char *scratch = nullptr;
    const int rc = scratch_address(&scratch);
    if (rc != HOUGH_OK)
        return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t blocks = (uint32_t)((n_bins + NA_ITEMS - 1) / NA_ITEMS);
    // the array keeps whatever the last call left in it: the ticket and the words this call will poll start at zero
    if (cudaMemsetAsync(scratch, 0, NA_HEAD_BYTES + (size_t)blocks * 8, st) != cudaSuccess) {
        (void)cudaGetLastError();
        return HOUGH_ECUDA;
    }
    NoallocParams p;
    p.acc = acc;
    p.n_bins = (uint32_t)n_bins;
    p.n_phi = n_phi;
    p.n_d0 = n_d0;
    p.n_kappa = n_kappa;
    p.L_min = L_min;
    p.wrap = phi_wrap;
    p.bin = bin;
    p.mask = mask;
    p.n_peaks = n_peaks;
    p.cap_peaks = cap_peaks;
    p.ticket = reinterpret_cast<unsigned int *>(scratch);
    p.status = reinterpret_cast<unsigned long long *>(scratch + NA_HEAD_BYTES);
    k_peaks_noalloc<<<blocks, NA_THREADS, 0, st>>>(p);
    return cudaGetLastError() == cudaSuccess ? HOUGH_OK : HOUGH_ECUDA;
}
