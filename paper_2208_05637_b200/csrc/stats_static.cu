// nqs_weighted_stats_static: the count-weighted statistics of Eq. 17 (counter :105) for callers that
// must not allocate device memory.
//
// Who that is.  A VMC driver usually hands the whole GPU to its framework's caching allocator (PyTorch's, or its own
// arena sized to the card) before the first iteration; a raw cudaMalloc issued by this library afterwards either fails,
// because nothing is left outside that pool, or takes memory the pool's bookkeeping does not know about and makes a
// later, legitimate request of the driver fail.  cudaMalloc / cudaFree also synchronise the whole device, which stalls
// the other streams of a loop that overlaps sampling, E_loc and the optimiser.  Processes confined to a fixed device
// memory budget (an MPS client with a pinned memory limit, a MIG slice shared by several ranks) are in the same
// position.  The other entry points of libnqs grow a workspace inside the model handle on demand; this one never does.
//
// How.  The kernel is the multi-CTA form of stats_kernel (kernels_simt.cu): every CTA reduces a slice of 2048 rows in
// fp64 in a fixed order and parks its four partial sums in scratch; the CTA that draws the last ticket adds the
// partials in CTA order and writes the caller's output.  The scratch is the file-scope array below — part of the
// library's device image, so every GPU that loads libnqs holds these 33 KB until the process exits — not an
// allocation.  Its address on a device is looked up once per device (cudaGetSymbolAddress) by the first call made
// with that device current.
#include <mutex>
#include "nqs_internal.h"

namespace {

constexpr int       SS_THREADS      = 256;
constexpr int       SS_ROWS_PER_THR = 8;
constexpr long long SS_ROWS_PER_CTA = (long long)SS_THREADS * SS_ROWS_PER_THR;      // 2048
constexpr int       SS_MAX_CTAS     = 1024;                                         // -> NQS_STATS_STATIC_MAX_ROWS rows
constexpr size_t    SS_PARTIAL_BYTES = sizeof(double) * 4 * SS_MAX_CTAS;            // 32 KB
constexpr size_t    SS_TICKET_OFFSET = SS_PARTIAL_BYTES;                            // one unsigned, on its own 256 B line
static_assert(SS_ROWS_PER_CTA * SS_MAX_CTAS == NQS_STATS_STATIC_MAX_ROWS, "header limit and scratch size disagree");

// [SS_MAX_CTAS][4] doubles of per-CTA partial sums, then the ticket counter.  In host code this NAME is only a handle
// for cudaGetSymbolAddress, never a pointer a kernel may be given: the kernel receives the address looked up on the
// device it is launched on.
static __device__ __align__(256) unsigned char g_stats_scratch[SS_PARTIAL_BYTES + 256];

__global__ void __launch_bounds__(SS_THREADS)
stats_static_kernel(const float2 *__restrict__ eloc, const long long *__restrict__ counts, long long B,
                    unsigned char *scratch, double *__restrict__ out4) {
    __shared__ double sh[4][SS_THREADS];
    __shared__ unsigned s_ticket;
    double *partial = (double *)scratch;
    unsigned *ticket = (unsigned *)(scratch + SS_TICKET_OFFSET);

    const long long base = (long long)blockIdx.x * SS_ROWS_PER_CTA;
    double a0 = 0, a1 = 0, a2 = 0, a3 = 0;
#pragma unroll
    for (int k = 0; k < SS_ROWS_PER_THR; ++k) {
        const long long i = base + threadIdx.x + (long long)k * SS_THREADS;
        if (i < B) {
            const double c = counts ? (double)counts[i] : 1.0;
            const float2 e = eloc[i];
            a0 += c; a1 += c * (double)e.x; a2 += c * (double)e.y;
            a3 += c * ((double)e.x * (double)e.x + (double)e.y * (double)e.y);
        }
    }
    sh[0][threadIdx.x] = a0; sh[1][threadIdx.x] = a1; sh[2][threadIdx.x] = a2; sh[3][threadIdx.x] = a3;
    __syncthreads();
    for (int s = SS_THREADS / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s)
            for (int q = 0; q < 4; ++q) sh[q][threadIdx.x] += sh[q][threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x < 4) {
        __stcg(&partial[4 * blockIdx.x + threadIdx.x], sh[threadIdx.x][0]);
        __threadfence();                               // the partial is visible device-wide before the ticket is drawn
    }
    __syncthreads();
    if (threadIdx.x == 0) s_ticket = atomicAdd(ticket, 1u);
    __syncthreads();
    if (s_ticket != gridDim.x - 1) return;
    // last CTA: every other CTA's partial is complete.  Sum in CTA order -> the result does not depend on scheduling.
    __threadfence();
    if (threadIdx.x < 4) {
        double s = 0;
        for (unsigned b = 0; b < gridDim.x; ++b) s += __ldcg(&partial[4 * b + threadIdx.x]);
        out4[threadIdx.x] = s;
    }
}

// Address of g_stats_scratch on each device, filled by that device's first call.
constexpr int SS_MAX_DEVICES = 64;
std::mutex g_setup_lock;
unsigned char *g_scratch_addr[SS_MAX_DEVICES] = {};

int scratch_for_current_device(unsigned char **out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return NQS_ECUDA; }
    if (dev < 0 || dev >= SS_MAX_DEVICES) return NQS_EUNSUPPORTED;
    std::lock_guard<std::mutex> guard(g_setup_lock);
    if (!g_scratch_addr[dev]) {
        const int rc = nqs_check_device();
        if (rc) return rc;
        unsigned char *p = nullptr;
        if (cudaGetSymbolAddress((void **)&p, g_stats_scratch) != cudaSuccess || !p) { cudaGetLastError(); return NQS_ECUDA; }
        g_scratch_addr[dev] = p;
    }
    *out = g_scratch_addr[dev];
    return NQS_OK;
}

}  // namespace

extern "C" int nqs_weighted_stats_static(const float *eloc_dev, const int64_t *counts_dev, int64_t B,
                                         double *stats_out_dev, void *cuda_stream) {
    if (B < 0 || !stats_out_dev || (B > 0 && !eloc_dev)) return NQS_EINVAL;
    if (B > NQS_STATS_STATIC_MAX_ROWS) return NQS_ERANGE;      // the scratch has one slot per 2048 rows, 1024 slots
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (B == 0) return cudaMemsetAsync(stats_out_dev, 0, 4 * sizeof(double), st) == cudaSuccess ? NQS_OK : NQS_ECUDA;
    unsigned char *scratch = nullptr;
    const int rc = scratch_for_current_device(&scratch);
    if (rc) return rc;
    // the array keeps whatever the previous call left: the ticket must start at zero, the partial slots are all
    // rewritten before they are read
    if (cudaMemsetAsync(scratch + SS_TICKET_OFFSET, 0, sizeof(unsigned), st) != cudaSuccess) { cudaGetLastError(); return NQS_ECUDA; }
    const unsigned grid = (unsigned)((B + SS_ROWS_PER_CTA - 1) / SS_ROWS_PER_CTA);
    stats_static_kernel<<<grid, SS_THREADS, 0, st>>>((const float2 *)eloc_dev, (const long long *)counts_dev, B, scratch,
                                                     stats_out_dev);
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? NQS_OK : NQS_ECUDA;
}
