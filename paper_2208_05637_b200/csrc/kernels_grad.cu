// Gradient of the energy objective, Eq. 7:
//     grad L = Re E[(l_theta(x) - b) conj(grad log f(x))],  b = E[l_theta],
// expectation over the unique samples weighted by their multiplicities, accumulated over
// gradient-accumulation mini-batches.  log f = log|psi| + i phi with two real networks, so the MADE
// parameters receive Re(E - b) through log|psi| and the phase-net parameters Im(E - b) through phi.
//
// The estimator needs grad log f only at the B SAMPLED rows (not at the B x G connected ones): 3 x the flops of B forward
// passes, ~1e-5 of the E_loc work at cfg 5.  It therefore runs on CUDA cores in fp32: a per-row kernel (forward pass +
// backward pass through the activations, 16 rows per CTA, activations in shared memory) that writes the layer inputs and
// the pre-activation gradients, and a tiled outer-product kernel that reduces them over the rows into the weight
// gradients (masked entries receive exactly 0: the ABI takes unmasked weights, include/nqs.h).  Everything is
// deterministic (fixed reduction order, no atomics).
#include <new>
#include "nqs_internal.h"

namespace {

constexpr int TR = 16;     // rows per CTA tile
constexpr int NT = 256;

__device__ __forceinline__ int bit128(ulonglong2 a, int q) { return (int)(((q < 64 ? a.x : a.y) >> (q & 63)) & 1ull); }

// out[j][r] = act(b[j] + sum_k Wt[k][j] in[k][r]); in/out smem tiles [.][TR]; Wt is [K][ldw] global (j contiguous)
template <bool RELU>
__device__ __forceinline__ void fwd(const float *__restrict__ Wt, int ldw, const float *__restrict__ bias, int K, int N,
                                    const float *in, float *out) {
    for (int j = threadIdx.x; j < N; j += NT) {
        float acc[TR];
        const float b = __ldg(bias + j);
#pragma unroll
        for (int r = 0; r < TR; ++r) acc[r] = b;
        for (int k = 0; k < K; ++k) {
            const float w = __ldg(Wt + (size_t)k * ldw + j);
#pragma unroll
            for (int r = 0; r < TR; r += 4) {
                const float4 a = *reinterpret_cast<const float4 *>(in + k * TR + r);
                acc[r] = fmaf(w, a.x, acc[r]); acc[r + 1] = fmaf(w, a.y, acc[r + 1]);
                acc[r + 2] = fmaf(w, a.z, acc[r + 2]); acc[r + 3] = fmaf(w, a.w, acc[r + 3]);
            }
        }
#pragma unroll
        for (int r = 0; r < TR; ++r) out[j * TR + r] = RELU ? fmaxf(acc[r], 0.0f) : acc[r];
    }
}

// din[k][r] = (post[k][r] > 0) * sum_j Wt[k][j] dout[j][r]   (transpose product through the same [in][out] array)
__device__ __forceinline__ void bwd(const float *__restrict__ Wt, int ldw, int K, int N, const float *dout, const float *post,
                                    float *din) {
    for (int k = threadIdx.x; k < K; k += NT) {
        float acc[TR];
#pragma unroll
        for (int r = 0; r < TR; ++r) acc[r] = 0.0f;
        const float *wrow = Wt + (size_t)k * ldw;
        for (int j = 0; j < N; ++j) {
            const float w = __ldg(wrow + j);
#pragma unroll
            for (int r = 0; r < TR; r += 4) {
                const float4 a = *reinterpret_cast<const float4 *>(dout + j * TR + r);
                acc[r] = fmaf(w, a.x, acc[r]); acc[r + 1] = fmaf(w, a.y, acc[r + 1]);
                acc[r + 2] = fmaf(w, a.z, acc[r + 2]); acc[r + 3] = fmaf(w, a.w, acc[r + 3]);
            }
        }
#pragma unroll
        for (int r = 0; r < TR; ++r) din[k * TR + r] = post[k * TR + r] > 0.0f ? acc[r] : 0.0f;
    }
}

// smem tile [dim][TR] -> global [row][ld] (dim contiguous), rows beyond `nrows` skipped
__device__ __forceinline__ void store_rows(const float *tile, int dim, float *g, int ld, long long row0, long long nrows) {
    for (int idx = threadIdx.x; idx < dim * TR; idx += NT) {
        const int r = idx / dim, j = idx % dim;
        if (row0 + r < nrows) g[(size_t)(row0 + r) * ld + j] = tile[j * TR + r];
    }
}

struct GradWs {      // per mini-batch, row-major [rows][dim]
    float *U, *X, *Y, *PH;           // layer inputs: [rows][npad], [rows][h] x 3
    float *dA, *dY, *dX, *dPH, *dO;  // pre-activation gradients: [rows][npad], [rows][h] x 3, [rows][4]
};

// stats3 = {sum n, sum n Re E, sum n Im E} over ALL samples (fp64, device): b = stats3[1..2] / stats3[0]
__global__ void __launch_bounds__(NT) grad_rows_kernel(MadeDev m, const ulonglong2 *__restrict__ x,
                                                       const long long *__restrict__ counts, const float2 *__restrict__ eloc,
                                                       const double *__restrict__ stats3, long long nrows, GradWs ws) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = m.n, h = m.h, npad = m.npad;
    float *U = reinterpret_cast<float *>(smem_raw);        // [npad][TR]
    float *X = U + (size_t)npad * TR;                      // [h][TR]
    float *Y = X + (size_t)h * TR;                         // [h][TR]
    float *T = Y + (size_t)h * TR;                         // [h][TR]
    float *A = T + (size_t)h * TR;                         // [npad][TR]
    float *O = A + (size_t)npad * TR;                      // [4][TR]
    float *wr = O + 4 * TR, *wi = wr + TR;                 // [TR] each
    __shared__ ulonglong2 cfg[TR];
    __shared__ ulonglong2 fmask[TR];                       // Eq. 14: clamped conditionals are constants -> no gradient through their logits
    const double tot = stats3[0], bre = stats3[1] / tot, bim = stats3[2] / tot;
    for (long long row0 = (long long)blockIdx.x * TR; row0 < nrows; row0 += (long long)gridDim.x * TR) {
        if (threadIdx.x < TR) {
            const long long i = row0 + threadIdx.x;
            if (i < nrows) {
                cfg[threadIdx.x] = x[i];
                const double c = counts ? (double)counts[i] : 1.0;
                const float2 e = eloc[i];
                wr[threadIdx.x] = (float)(c * ((double)e.x - bre) / tot);
                wi[threadIdx.x] = (float)(c * ((double)e.y - bim) / tot);
            } else { cfg[threadIdx.x] = make_ulonglong2(0, 0); wr[threadIdx.x] = 0.f; wi[threadIdx.x] = 0.f; }
        }
        __syncthreads();
        for (int idx = threadIdx.x; idx < npad * TR; idx += NT) {
            const int d = idx / TR, r = idx % TR;
            U[idx] = d < n ? (bit128(cfg[r], __ldg(m.order + d)) ? 1.0f : -1.0f) : 0.0f;
        }
        if (threadIdx.x < TR) {
            ulonglong2 f = make_ulonglong2(0, 0);
            if (m.n_up >= 0) {
                const int r = threadIdx.x;
                ulonglong2 zp = make_ulonglong2(0, 0);
                for (int d = 0; d < n; ++d)
                    if (bit128(cfg[r], __ldg(m.order + d))) { if (d < 64) zp.x |= 1ull << d; else zp.y |= 1ull << (d - 64); }
                bool valid;
                f = nqs_forced_mask(zp, n, m.spin_lo, m.spin_hi, m.n_up, m.n_down, &valid);
            }
            fmask[threadIdx.x] = f;
        }
        __syncthreads();
        store_rows(U, npad, ws.U, npad, row0, nrows);
        // ---- modulus net forward ----
        fwd<true>(m.w1t, h, m.b1, n, h, U, X);
        __syncthreads();
        store_rows(X, h, ws.X, h, row0, nrows);
        const float *hid = X;
        if (m.L == 2) {
            fwd<true>(m.w2t, h, m.b2, h, h, X, Y);
            __syncthreads();
            store_rows(Y, h, ws.Y, h, row0, nrows);
            hid = Y;
        }
        fwd<false>(m.w3t, npad, m.b3, h, npad, hid, A);
        __syncthreads();
        // dA[d][r] = wr_r * 1/2 * s * sigmoid(-s a),  s = +-1 = U  (d/da log sigmoid(s a) = s sigmoid(-s a))
        for (int idx = threadIdx.x; idx < npad * TR; idx += NT) {
            const int d = idx / TR, r = idx % TR;
            const float s = U[idx], a = A[idx];
            const bool clamped = ((d < 64 ? fmask[r].x : fmask[r].y) >> (d & 63)) & 1ull;
            A[idx] = (d < n && !clamped) ? wr[r] * 0.5f * s / (1.0f + expf(s * a)) : 0.0f;
        }
        __syncthreads();
        store_rows(A, npad, ws.dA, npad, row0, nrows);
        // ---- backward through the hidden layers ----
        if (m.L == 2) {
            bwd(m.w3t, npad, h, npad, A, Y, T);                 // dY (pre-activation) in T
            __syncthreads();
            store_rows(T, h, ws.dY, h, row0, nrows);
            bwd(m.w2t, h, h, h, T, X, Y);                       // dX (pre-activation) in Y
            __syncthreads();
            store_rows(Y, h, ws.dX, h, row0, nrows);
        } else {
            bwd(m.w3t, npad, h, npad, A, X, T);                 // dX in T
            __syncthreads();
            store_rows(T, h, ws.dX, h, row0, nrows);
        }
        __syncthreads();
        // ---- phase net: forward, then backward of wi * o[sel] ----
        fwd<true>(m.p1t, h, m.c1, n, h, U, X);                  // p1t rows n-2, n-1 are zero: the last two inputs do not enter
        __syncthreads();
        store_rows(X, h, ws.PH, h, row0, nrows);
        if (threadIdx.x < 4 * TR) {
            const int o = threadIdx.x / TR, r = threadIdx.x % TR;
            const int sel = (U[(n - 2) * TR + r] > 0.0f ? 2 : 0) + (U[(n - 1) * TR + r] > 0.0f ? 1 : 0);
            O[o * TR + r] = o == sel ? wi[r] : 0.0f;
        }
        __syncthreads();
        store_rows(O, 4, ws.dO, 4, row0, nrows);
        bwd(m.p2t, 4, h, 4, O, X, T);                           // dPH in T
        __syncthreads();
        store_rows(T, h, ws.dPH, h, row0, nrows);
        __syncthreads();
    }
}

// out[i][j] += mask(i, j) * sum_r dZ[r][i] * act[r][j],  mask = rowdeg[i] >= coldeg[j] (NULL = no mask);
// optionally bias[i] += sum_r dZ[r][i] (blockIdx.y == 0).  One CTA per 64 x 64 output tile, fixed order over r.
constexpr int WT = 64, WK = 16;
__global__ void __launch_bounds__(256) wgrad_kernel(const float *__restrict__ dZ, int ldz, const float *__restrict__ act, int lda,
                                                    long long rows, int M, int N, const int *__restrict__ rowdeg,
                                                    const int *__restrict__ coldeg, float *__restrict__ out, int ldo,
                                                    float *__restrict__ bias_out) {
    __shared__ float sA[WK][WT + 1], sB[WK][WT + 1];
    const int i0 = blockIdx.x * WT, j0 = blockIdx.y * WT;
    const int ti = threadIdx.x / 16, tj = threadIdx.x % 16;       // 16 x 16 threads, 4 x 4 outputs each
    float acc[4][4] = {};
    float bsum = 0.0f;                                            // threads 0..63 of blockIdx.y == 0: column sums of dZ
    for (long long r0 = 0; r0 < rows; r0 += WK) {
        for (int idx = threadIdx.x; idx < WK * WT; idx += 256) {
            const int r = idx / WT, c = idx % WT;
            const bool rv = r0 + r < rows;
            sA[r][c] = (rv && i0 + c < M) ? dZ[(size_t)(r0 + r) * ldz + i0 + c] : 0.0f;
            sB[r][c] = (rv && j0 + c < N) ? act[(size_t)(r0 + r) * lda + j0 + c] : 0.0f;
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < WK; ++r) {
            float a[4], b[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) { a[q] = sA[r][ti * 4 + q]; b[q] = sB[r][tj * 4 + q]; }
#pragma unroll
            for (int p = 0; p < 4; ++p)
#pragma unroll
                for (int q = 0; q < 4; ++q) acc[p][q] = fmaf(a[p], b[q], acc[p][q]);
        }
        if (bias_out && blockIdx.y == 0 && threadIdx.x < WT) {
#pragma unroll
            for (int r = 0; r < WK; ++r) bsum += sA[r][threadIdx.x];
        }
        __syncthreads();
    }
#pragma unroll
    for (int p = 0; p < 4; ++p)
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int i = i0 + ti * 4 + p, j = j0 + tj * 4 + q;
            if (i < M && j < N) {
                const bool keep = !rowdeg || rowdeg[i] >= coldeg[j];
                if (keep) out[(size_t)i * ldo + j] += acc[p][q];
            }
        }
    if (bias_out && blockIdx.y == 0 && threadIdx.x < WT && i0 + (int)threadIdx.x < M) bias_out[i0 + threadIdx.x] += bsum;
}

// {sum n, sum n Re E, sum n Im E} in fp64, one CTA, fixed order
__global__ void __launch_bounds__(256) grad_stats_kernel(const float2 *__restrict__ eloc, const long long *__restrict__ counts,
                                                         long long B, double *__restrict__ out3) {
    __shared__ double sh[3][256];
    double a0 = 0, a1 = 0, a2 = 0;
    for (long long i = threadIdx.x; i < B; i += 256) {
        const double c = counts ? (double)counts[i] : 1.0;
        const float2 e = eloc[i];
        a0 += c; a1 += c * (double)e.x; a2 += c * (double)e.y;
    }
    sh[0][threadIdx.x] = a0; sh[1][threadIdx.x] = a1; sh[2][threadIdx.x] = a2;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) for (int q = 0; q < 3; ++q) sh[q][threadIdx.x] += sh[q][threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x < 3) out3[threadIdx.x] = sh[threadIdx.x][0];
}

}  // namespace

struct GradPack {
    void *d_deg = nullptr;        // int32: [rowdeg/coldeg arrays, see offsets below]
    int off_in = 0, off_h[2] = {0, 0}, off_hp1[2] = {0, 0}, off_out = 0;   // d+1 | deg_k | deg_k + 1 | d+1
    void *ws = nullptr; size_t ws_bytes = 0;
    void *d_stats = nullptr;
};

void grad_pack_free(const nqs_made *M) {
    if (!M->grad) return;
    cudaFree(M->grad->d_deg); cudaFree(M->grad->ws); cudaFree(M->grad->d_stats);
    delete M->grad;
    M->grad = nullptr;
}

static int grad_pack(const nqs_made *M) {
    if (M->grad) return NQS_OK;
    GradPack *G = new (std::nothrow) GradPack();
    if (!G) return NQS_ENOMEM;
    const int n = M->n, h = M->h, L = M->L;
    std::vector<int32_t> deg;
    G->off_in = 0;
    for (int d = 0; d < n; ++d) deg.push_back(d + 1);                              // m_in[d] = d + 1
    for (int k = 0; k < L; ++k) { G->off_h[k] = (int)deg.size(); for (int j = 0; j < h; ++j) deg.push_back(M->deg[(size_t)k * h + j]); }
    for (int k = 0; k < L; ++k) { G->off_hp1[k] = (int)deg.size(); for (int j = 0; j < h; ++j) deg.push_back(M->deg[(size_t)k * h + j] + 1); }
    if (cudaMalloc(&G->d_deg, deg.size() * 4) != cudaSuccess || cudaMalloc(&G->d_stats, 64) != cudaSuccess ||
        cudaMemcpy(G->d_deg, deg.data(), deg.size() * 4, cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        cudaFree(G->d_deg); cudaFree(G->d_stats);
        delete G;
        return NQS_ECUDA;
    }
    M->grad = G;
    return NQS_OK;
}

extern "C" int nqs_made_num_params(const nqs_made_t *M, int64_t *n_params) {
    if (!M || !n_params) return NQS_EINVAL;
    const int64_t n = M->n, h = M->h, L = M->L;
    int64_t t = h * n + h + n * h + n + h * (n - 2) + h + 4 * h + 4;
    if (L == 2) t += h * h + h;
    *n_params = t;
    return NQS_OK;
}

static inline size_t al256(size_t x) { return (x + 255) & ~(size_t)255; }

extern "C" int nqs_energy_grad(const nqs_made_t *M, const uint64_t *samples_dev, const int64_t *counts_dev,
                               const float *eloc_dev, int64_t B, int64_t minibatch, const double *global_stats_host,
                               float *grad_out_dev, double *baseline_out_host, void *cuda_stream) {
    if (!M || B < 0 || minibatch < 0 || !grad_out_dev) return NQS_EINVAL;
    if (B > 0 && (!samples_dev || !eloc_dev)) return NQS_EINVAL;
    int rc = nqs_made_upload(M);
    if (rc) return rc;
    if ((rc = grad_pack(M))) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t smem = sizeof(float) * ((size_t)(2 * M->npad + 3 * M->h + 4 + 2) * TR);
    if (smem > 227 * 1024) return NQS_EUNSUPPORTED;                 // before anything is enqueued
    if (global_stats_host && !(global_stats_host[0] > 0.0)) return NQS_EINVAL;
    int64_t np = 0;
    nqs_made_num_params(M, &np);
    if (cudaMemsetAsync(grad_out_dev, 0, sizeof(float) * (size_t)np, st) != cudaSuccess) return NQS_ECUDA;
    if (B == 0) {
        if (baseline_out_host) baseline_out_host[0] = baseline_out_host[1] = 0.0;
        return NQS_OK;
    }
    GradPack *G = M->grad;
    const int n = M->n, h = M->h, L = M->L, npad = M->npad;
    const long long mb = minibatch > 0 ? minibatch : 8192;
    const long long mbe = mb < B ? mb : B;
    // workspace: U, dA [mbe][npad]; X, Y, PH, dY, dX, dPH [mbe][h]; dO [mbe][4]
    const size_t s_np = al256(sizeof(float) * (size_t)mbe * npad), s_h = al256(sizeof(float) * (size_t)mbe * h), s_4 = al256(sizeof(float) * (size_t)mbe * 4);
    const size_t need = 2 * s_np + 6 * s_h + s_4;
    if (G->ws_bytes < need) {
        if (G->ws) cudaFree(G->ws);
        G->ws = nullptr; G->ws_bytes = 0;
        if (cudaMalloc(&G->ws, need) != cudaSuccess) { cudaGetLastError(); return NQS_ENOMEM; }
        G->ws_bytes = need;
    }
    unsigned char *w = (unsigned char *)G->ws;
    GradWs ws;
    ws.U = (float *)w; w += s_np; ws.dA = (float *)w; w += s_np;
    ws.X = (float *)w; w += s_h; ws.Y = (float *)w; w += s_h; ws.PH = (float *)w; w += s_h;
    ws.dY = (float *)w; w += s_h; ws.dX = (float *)w; w += s_h; ws.dPH = (float *)w; w += s_h;
    ws.dO = (float *)w;
    double *d_stats = (double *)G->d_stats;
    if (global_stats_host) {          // data-parallel replicas: {sum n, sum n Re E, sum n Im E} over ALL ranks' samples
        if (cudaMemcpyAsync(d_stats, global_stats_host, 3 * sizeof(double), cudaMemcpyHostToDevice, st) != cudaSuccess) return NQS_ECUDA;
    } else {
        grad_stats_kernel<<<1, 256, 0, st>>>((const float2 *)eloc_dev, (const long long *)counts_dev, B, d_stats);
        ++g_launch_count;
    }
    if (cudaFuncSetAttribute(grad_rows_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) { cudaGetLastError(); return NQS_ECUDA; }
    int sms = 148, dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    // flat gradient layout (include/nqs.h): W_0, b_0, (W_1, b_1,) W_L, b_L, P1, c1, P2, c2
    float *g = grad_out_dev;
    float *gW0 = g; g += (size_t)h * n; float *gb0 = g; g += h;
    float *gW1 = nullptr, *gb1 = nullptr;
    if (L == 2) { gW1 = g; g += (size_t)h * h; gb1 = g; g += h; }
    float *gWo = g; g += (size_t)n * h; float *gbo = g; g += n;
    float *gP1 = g; g += (size_t)h * (n - 2); float *gc1 = g; g += h;
    float *gP2 = g; g += (size_t)4 * h; float *gc2 = g;
    const int *deg = (const int *)G->d_deg;
    auto wgrad = [&](const float *dZ, int ldz, const float *act, int lda, long long rows, int Mo, int No, const int *rd, const int *cd,
                     float *out, float *bout) {
        dim3 grid((unsigned)((Mo + WT - 1) / WT), (unsigned)((No + WT - 1) / WT));
        wgrad_kernel<<<grid, 256, 0, st>>>(dZ, ldz, act, lda, rows, Mo, No, rd, cd, out, No, bout);
        ++g_launch_count;
    };
    for (long long i0 = 0; i0 < B; i0 += mb) {                       // gradient accumulation
        const long long nb = (B - i0 < mb) ? (B - i0) : mb;
        const long long ntile = (nb + TR - 1) / TR;
        const int grid = (int)(ntile < (long long)sms * 2 ? ntile : (long long)sms * 2);
        grad_rows_kernel<<<grid, NT, smem, st>>>(M->dev, (const ulonglong2 *)samples_dev + i0,
                                                 counts_dev ? (const long long *)counts_dev + i0 : nullptr,
                                                 (const float2 *)eloc_dev + i0, d_stats, nb, ws);
        ++g_launch_count;
        // masks (include/nqs.h): M1[j][d] = deg_0[j] >= d+1; Mk[j'][j] = deg_k[j'] >= deg_{k-1}[j]; Mout[d][j] = d+1 >= deg_L[j] + 1
        wgrad(ws.dX, h, ws.U, npad, nb, h, n, deg + G->off_h[0], deg + G->off_in, gW0, gb0);
        if (L == 2) wgrad(ws.dY, h, ws.X, h, nb, h, h, deg + G->off_h[1], deg + G->off_h[0], gW1, gb1);
        wgrad(ws.dA, npad, L == 2 ? ws.Y : ws.X, h, nb, n, h, deg + G->off_in, deg + G->off_hp1[L - 1], gWo, gbo);
        wgrad(ws.dPH, h, ws.U, npad, nb, h, n - 2, nullptr, nullptr, gP1, gc1);
        wgrad(ws.dO, 4, ws.PH, h, nb, 4, h, nullptr, nullptr, gP2, gc2);
    }
    if (cudaGetLastError() != cudaSuccess) return NQS_ECUDA;
    if (baseline_out_host) {
        double s3[3];
        if (cudaMemcpyAsync(s3, d_stats, sizeof(s3), cudaMemcpyDeviceToHost, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) return NQS_ECUDA;
        baseline_out_host[0] = s3[1] / s3[0]; baseline_out_host[1] = s3[2] / s3[0];
    }
    return NQS_OK;
}
