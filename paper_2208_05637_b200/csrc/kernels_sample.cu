// Batched autoregressive sampler, PAPER.md:105-107 and :136-142 (Eq. 14): a buffer of unique prefixes with occurrence
// counters, doubled at every autoregressive position, counters split by Bernoulli trials with the conditionals of a
// forward pass on the buffer, lowest counters eliminated.  Readings (A13 / A25, same as oracle/sampler.py —
// written independently of it): the split of a counter of c occurrences is c Bernoulli trials, one per DRAW; draw s at
// position d uses u = (w + 1/2) 2^-32, w = first word of Philox4x32-10(key = seed, counter = (s, d)), and takes bit 1
// iff u < pi_hat; children of buffer entry i sit at 2i, 2i + 1; zero counters leave; above `max_unique` the largest
// counters stay (ties: buffer order) and the dropped draws are discarded.
// The conditionals come from the fp32 CUDA-core forward (cond_kernel, kernels_simt.cu): n sequential sweeps over at most
// max_unique rows, ~1e-4 of the E_loc work.
#include "nqs_internal.h"

namespace {

__device__ __forceinline__ uint32_t philox_first_word(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return c0;
}

// one Bernoulli trial per live draw: entry[t] <- child index 2 e + bit, ccount[child] += 1
__global__ void draw_kernel(int *__restrict__ entry, long long n_draws, int d, unsigned long long seed,
                            const float *__restrict__ p1, unsigned long long *__restrict__ ccount) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_draws) return;
    const int e = entry[t];
    if (e < 0) return;                                          // draw discarded by an earlier elimination
    const uint32_t w = philox_first_word((uint32_t)t, (uint32_t)((unsigned long long)t >> 32), (uint32_t)d, 0u,
                                         (uint32_t)seed, (uint32_t)(seed >> 32));
    const double u = ((double)w + 0.5) * 2.3283064365386963e-10;      // 2^-32
    const int child = 2 * e + (u < (double)p1[e] ? 1 : 0);
    entry[t] = child;
    atomicAdd(&ccount[child], 1ull);
}

// Stable compaction of the doubled buffer with elimination of the lowest counters.  One CTA of 1024 threads, each
// owning a contiguous chunk of children.  keep(c) = count > 0 when at most `cap` children are non-zero (or cap == 0);
// otherwise the cap largest counters, ties broken by buffer order: with T the cap-th largest counter value, every child
// with count > T and the first cap - #(count > T) children with count == T.  newidx[c] = position in the new buffer or -1.
constexpr int CT = 1024;

__device__ long long block_sum(long long v, long long *sh) {
    sh[threadIdx.x] = v;
    __syncthreads();
    for (int s = CT / 2; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    const long long r = sh[0];
    __syncthreads();
    return r;
}

// exclusive prefix over the per-thread values (fixed order)
__device__ long long block_excl_scan(long long v, long long *sh) {
    sh[threadIdx.x] = v;
    __syncthreads();
    for (int off = 1; off < CT; off <<= 1) {
        const long long add = (int)threadIdx.x >= off ? sh[threadIdx.x - off] : 0;
        __syncthreads();
        sh[threadIdx.x] += add;
        __syncthreads();
    }
    const long long r = sh[threadIdx.x] - v;
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(CT) compact_kernel(const unsigned long long *__restrict__ ccount, long long nchild, long long cap,
                                                     int *__restrict__ newidx, long long *__restrict__ n_new) {
    __shared__ long long sh[CT];
    const long long chunk = (nchild + CT - 1) / CT;
    const long long lo = (long long)threadIdx.x * chunk, hi = lo + chunk < nchild ? lo + chunk : nchild;
    long long nz = 0;
    unsigned long long mx = 0;
    for (long long c = lo; c < hi; ++c) { const unsigned long long v = ccount[c]; nz += v > 0; mx = v > mx ? v : mx; }
    const long long nnz = block_sum(nz, sh);
    unsigned long long T = 0;                 // keep count > T, plus `quota` ties at count == T (T == 0: keep every non-zero child)
    long long quota = 0;
    if (cap > 0 && nnz > cap) {
        // largest counter over the block
        sh[threadIdx.x] = (long long)mx;
        __syncthreads();
        for (int s = CT / 2; s > 0; s >>= 1) {
            if ((int)threadIdx.x < s && sh[threadIdx.x + s] > sh[threadIdx.x]) sh[threadIdx.x] = sh[threadIdx.x + s];
            __syncthreads();
        }
        unsigned long long tlo = 1, thi = (unsigned long long)sh[0] + 1;      // f(tlo) >= cap > f(thi), f(t) = #(count >= t)
        __syncthreads();
        while (thi - tlo > 1) {
            const unsigned long long mid = tlo + (thi - tlo) / 2;
            long long ge = 0;
            for (long long c = lo; c < hi; ++c) ge += ccount[c] >= mid;
            if (block_sum(ge, sh) >= cap) tlo = mid; else thi = mid;
        }
        T = tlo;
        long long gt = 0;
        for (long long c = lo; c < hi; ++c) gt += ccount[c] > T;
        quota = cap - block_sum(gt, sh);
    }
    // ties before this thread's chunk, then kept children before it
    long long eq = 0;
    if (T > 0) for (long long c = lo; c < hi; ++c) eq += ccount[c] == T;
    long long eq_before = T > 0 ? block_excl_scan(eq, sh) : 0;
    long long kept = 0, e2 = eq_before;
    for (long long c = lo; c < hi; ++c) {
        const unsigned long long v = ccount[c];
        bool k;
        if (T == 0) k = v > 0; else { k = v > T || (v == T && e2 < quota); e2 += v == T; }
        kept += k;
    }
    long long pos = block_excl_scan(kept, sh);
    e2 = eq_before;
    for (long long c = lo; c < hi; ++c) {
        const unsigned long long v = ccount[c];
        bool k;
        if (T == 0) k = v > 0; else { k = v > T || (v == T && e2 < quota); e2 += v == T; }
        newidx[c] = k ? (int)pos++ : -1;
    }
    const long long total = block_sum(kept, sh);
    if (threadIdx.x == 0) *n_new = total;
}

// new buffer: entry newidx[c] = parent c / 2 with bit (c & 1) written at the qubit of this position
__global__ void build_kernel(const ulonglong2 *__restrict__ cfg, const unsigned long long *__restrict__ ccount,
                             const int *__restrict__ newidx, long long nchild, int qubit, ulonglong2 *__restrict__ cfg_new,
                             long long *__restrict__ counts_new) {
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= nchild) return;
    const int ni = newidx[c];
    if (ni < 0) return;
    ulonglong2 v = cfg[c >> 1];
    if (c & 1) { if (qubit < 64) v.x |= 1ull << qubit; else v.y |= 1ull << (qubit - 64); }
    cfg_new[ni] = v;
    counts_new[ni] = (long long)ccount[c];
}

__global__ void remap_kernel(int *__restrict__ entry, long long n_draws, const int *__restrict__ newidx) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_draws) return;
    const int e = entry[t];
    if (e >= 0) entry[t] = newidx[e];
}

}  // namespace

extern "C" int nqs_made_sample(const nqs_made_t *M, int64_t n_draws, uint64_t seed, int n_up, int n_down,
                               int64_t max_unique, uint64_t *samples_out_dev, int64_t *counts_out_dev,
                               int64_t *n_unique_out_host, void *cuda_stream) {
    if (!M || n_draws < 0 || max_unique < 0 || !n_unique_out_host) return NQS_EINVAL;
    if (n_draws > 0 && (!samples_out_dev || !counts_out_dev)) return NQS_EINVAL;
    if (n_draws > 0x7FFFFFFFll / 2) return NQS_ERANGE;            // buffer indices are 32-bit
    const int n = M->n;
    if ((n_up < 0) != (n_down < 0)) return NQS_EINVAL;
    // One model, one distribution: when the handle carries a constraint (nqs_made_set_constraint) the samples must
    // come from the same pi_hat that log psi, E_loc and the gradient use.  (-1, -1) takes the handle's; a different
    // pair is a caller's mistake, not a request.
    if (M->n_up >= 0) {
        if (n_up < 0) { n_up = M->n_up; n_down = M->n_down; }
        else if (n_up != M->n_up || n_down != M->n_down) return NQS_EINVAL;
    }
    if (n_up >= 0) {                                              // Eq. 12: even qubits hold the up spins, odd qubits the down spins
        if (n_up > (n + 1) / 2 || n_down > n / 2) return NQS_EINVAL;
    }
    *n_unique_out_host = 0;
    if (n_draws == 0) return NQS_OK;
    int rc = nqs_made_upload(M);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long emax = max_unique > 0 && max_unique < n_draws ? max_unique : n_draws;     // buffer entries after a step
    // buffers: one arena in the model handle, grown on demand and kept (a handle serves one call at a time), so a
    // training loop that samples every iteration allocates on its first iteration only
    auto al = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const size_t sz_cfg = al(16 * (size_t)emax), sz_cnt = al(8 * (size_t)emax), sz_cc = al(16 * (size_t)emax),
                 sz_ni = al(8 * (size_t)emax), sz_entry = al(4 * (size_t)n_draws), sz_p1 = al(4 * (size_t)emax), sz_n = 256;
    const size_t need = 2 * sz_cfg + sz_cnt + sz_cc + sz_ni + sz_entry + sz_p1 + sz_n;
    if (M->samp_ws_bytes < need) {
        if (M->samp_ws) cudaFree(M->samp_ws);
        M->samp_ws = nullptr; M->samp_ws_bytes = 0;
        if (cudaMalloc(&M->samp_ws, need) != cudaSuccess) { cudaGetLastError(); return NQS_ENOMEM; }
        M->samp_ws_bytes = need;
    }
    unsigned char *wsp = (unsigned char *)M->samp_ws;
    void *d_cfg[2];
    d_cfg[0] = wsp; wsp += sz_cfg; d_cfg[1] = wsp; wsp += sz_cfg;
    void *d_cnt = wsp; wsp += sz_cnt;
    void *d_cc = wsp; wsp += sz_cc;
    void *d_ni = wsp; wsp += sz_ni;
    void *d_entry = wsp; wsp += sz_entry;
    void *d_p1 = wsp; wsp += sz_p1;
    void *d_n = wsp;
    rc = NQS_ECUDA;
    long long E = 1;
    int cur = 0;
    bool ok = cudaMemsetAsync(d_cfg[0], 0, 16, st) == cudaSuccess && cudaMemsetAsync(d_entry, 0, 4 * (size_t)n_draws, st) == cudaSuccess;
    for (int d = 0; ok && d < n; ++d) {
        // forward pass on the buffer: pi_hat(z_d = 1 | prefix) with the Eq. 14 clamp
        int r2 = launch_cond_simt(M->dev, (const ulonglong2 *)d_cfg[cur], E, d, n_up, n_down, (float *)d_p1, st);
        if (r2) { rc = r2; ok = false; break; }
        const long long nchild = 2 * E;
        ok = cudaMemsetAsync(d_cc, 0, 8 * (size_t)nchild, st) == cudaSuccess;
        if (!ok) break;
        draw_kernel<<<(unsigned)((n_draws + 255) / 256), 256, 0, st>>>((int *)d_entry, n_draws, d, seed, (const float *)d_p1,
                                                                        (unsigned long long *)d_cc);
        compact_kernel<<<1, CT, 0, st>>>((const unsigned long long *)d_cc, nchild, max_unique, (int *)d_ni, (long long *)d_n);
        build_kernel<<<(unsigned)((nchild + 255) / 256), 256, 0, st>>>((const ulonglong2 *)d_cfg[cur], (const unsigned long long *)d_cc,
                                                                        (const int *)d_ni, nchild, M->order[d],
                                                                        (ulonglong2 *)d_cfg[cur ^ 1], (long long *)d_cnt);
        remap_kernel<<<(unsigned)((n_draws + 255) / 256), 256, 0, st>>>((int *)d_entry, n_draws, (const int *)d_ni);
        g_launch_count += 4;
        long long enew = 0;
        ok = cudaMemcpyAsync(&enew, d_n, 8, cudaMemcpyDeviceToHost, st) == cudaSuccess && cudaStreamSynchronize(st) == cudaSuccess &&
             cudaGetLastError() == cudaSuccess;
        if (ok && (enew < 1 || enew > emax)) { ok = false; }
        E = enew;
        cur ^= 1;
    }
    if (ok) {
        ok = cudaMemcpyAsync(samples_out_dev, d_cfg[cur], 16 * (size_t)E, cudaMemcpyDeviceToDevice, st) == cudaSuccess &&
             cudaMemcpyAsync(counts_out_dev, d_cnt, 8 * (size_t)E, cudaMemcpyDeviceToDevice, st) == cudaSuccess &&
             cudaStreamSynchronize(st) == cudaSuccess;
    }
    if (!ok) { cudaGetLastError(); return rc; }
    *n_unique_out_host = E;
    return NQS_OK;
}
