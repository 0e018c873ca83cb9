// CUDA-core (fp32 FFMA) kernels: MADE forward, Pauli contraction, fused local energy, statistics.
// This is the reference-quality CUDA path (NQS_PATH_SIMT): any shape, fp32 end to end.  The tensor-core
// path lives in kernels_tc.cu; the contraction / statistics kernels here are shared by both.
#include <cstdio>
#include "nqs_internal.h"

namespace {

constexpr int TR = 16;     // rows (configurations) per CTA tile
constexpr int NT = 256;    // threads per CTA

__device__ __forceinline__ int bit128(ulonglong2 a, int q) {
    return (int)(((q < 64 ? a.x : a.y) >> (q & 63)) & 1ull);
}

// log sigmoid(t) = min(t,0) - log1p(exp(-|t|))
__device__ __forceinline__ float log_sigmoid(float t) { return fminf(t, 0.0f) - log1pf(expf(-fabsf(t))); }

// out[j][r] = act(b[j] + sum_k Wt[k][j] * in[k][r]),  in/out are smem tiles [.][TR]; Wt is [K][ldw] global.
// Work item = (output j, group of RPT rows); items are strided over the CTA.  kend (or NULL): output j has no non-zero
// weight at k >= kend[j] (masked layers), so the sum stops there — exact, the skipped terms are w = 0.
template <int RPT, bool RELU>
__device__ __forceinline__ void layer_fwd(const float *__restrict__ Wt, int ldw, const float *__restrict__ bias,
                                          int K, int N, const float *in, float *out, const int32_t *__restrict__ kend = nullptr) {
    constexpr int RG = TR / RPT;
    for (int item = threadIdx.x; item < N * RG; item += NT) {
        const int j = item % N, rg = item / N;
        float acc[RPT];
        const float b = __ldg(bias + j);
#pragma unroll
        for (int r = 0; r < RPT; ++r) acc[r] = b;
        const float *inp = in + rg * RPT;
        const int kstop = kend ? min(K, __ldg(kend + j)) : K;
#pragma unroll 4
        for (int k = 0; k < kstop; ++k) {
            const float w = __ldg(Wt + (size_t)k * ldw + j);
            if constexpr (RPT >= 4) {
#pragma unroll
                for (int r = 0; r < RPT; r += 4) {
                    const float4 a = *reinterpret_cast<const float4 *>(inp + k * TR + r);
                    acc[r] = fmaf(w, a.x, acc[r]);
                    acc[r + 1] = fmaf(w, a.y, acc[r + 1]);
                    acc[r + 2] = fmaf(w, a.z, acc[r + 2]);
                    acc[r + 3] = fmaf(w, a.w, acc[r + 3]);
                }
            } else {
#pragma unroll
                for (int r = 0; r < RPT; ++r) acc[r] = fmaf(w, inp[k * TR + r], acc[r]);
            }
        }
#pragma unroll
        for (int r = 0; r < RPT; ++r) out[j * TR + rg * RPT + r] = RELU ? fmaxf(acc[r], 0.0f) : acc[r];
    }
}

struct Smem {
    float *U, *X, *Y, *A, *O, *red;   // [n][TR], [h][TR], [h][TR], [npad][TR], [4][TR], [16][TR]
    ulonglong2 *cfg;                  // [TR]
    float *lp, *phi;                  // [TR]
    float *keep;                      // [npad][TR]: 0 where Eq. 14 clamps the conditional (constraint on), else 1
    float *bad;                       // [TR]: 1 if the row violates Eq. 12 (psi = 0)
};

__device__ __forceinline__ Smem carve(unsigned char *base, const MadeDev &m) {
    Smem s;
    float *p = reinterpret_cast<float *>(base);
    s.cfg = reinterpret_cast<ulonglong2 *>(p); p += TR * 4;
    s.U = p; p += (size_t)m.npad * TR;
    s.X = p; p += (size_t)m.h * TR;
    s.Y = p; p += (size_t)m.h * TR;
    s.A = p; p += (size_t)m.npad * TR;
    s.O = p; p += 4 * TR;
    s.red = p; p += 16 * TR;
    s.lp = p; p += TR;
    s.phi = p; p += TR;
    s.keep = p; p += (size_t)m.npad * TR;
    s.bad = p; p += TR;
    return s;
}

size_t smem_bytes(const MadeDev &m) {
    return sizeof(float) * ((size_t)TR * 4 + 3 * (size_t)m.npad * TR + 2 * (size_t)m.h * TR + 4 * TR + 16 * TR + 3 * TR);
}

// MADE + phase forward for the TR configurations in s.cfg -> s.lp[r] = log|psi|, s.phi[r] = phi.
// PAPER.md:84 (layers), :96 Eq. 10.  All threads of the CTA must call; ends with a __syncthreads().
__device__ void forward_tile(const MadeDev &m, const Smem &s) {
    const int n = m.n, h = m.h;
    // inputs u_d = 2 z_d - 1 with z_d = bit order[d]  (position order)
    for (int idx = threadIdx.x; idx < n * TR; idx += NT) {
        const int d = idx / TR, r = idx % TR;
        s.U[idx] = bit128(s.cfg[r], __ldg(m.order + d)) ? 1.0f : -1.0f;
    }
    if (m.n_up >= 0 && threadIdx.x < TR) {                      // Eq. 14: which conditionals are clamped for this row
        const int r = threadIdx.x;
        ulonglong2 zp = make_ulonglong2(0, 0);
        for (int d = 0; d < n; ++d)
            if (bit128(s.cfg[r], __ldg(m.order + d))) { if (d < 64) zp.x |= 1ull << d; else zp.y |= 1ull << (d - 64); }
        bool valid;
        const ulonglong2 fm = nqs_forced_mask(zp, n, m.spin_lo, m.spin_hi, m.n_up, m.n_down, &valid);
        for (int d = 0; d < n; ++d) s.keep[d * TR + r] = ((d < 64 ? fm.x : fm.y) >> (d & 63)) & 1ull ? 0.0f : 1.0f;
        s.bad[r] = valid ? 0.0f : 1.0f;
    }
    __syncthreads();
    layer_fwd<TR, true>(m.w1t, h, m.b1, n, h, s.U, s.X, m.kend1);
    __syncthreads();
    const float *hid = s.X;
    if (m.L == 2) {
        layer_fwd<TR, true>(m.w2t, h, m.b2, h, h, s.X, s.Y, m.kend2);
        __syncthreads();
        hid = s.Y;
    }
    layer_fwd<4, false>(m.w3t, m.npad, m.b3, h, n, hid, s.A, m.kend3);
    float *ph = (m.L == 2) ? s.X : s.Y;                 // a free [h][TR] buffer
    __syncthreads();                                     // (L==2: X no longer read by layer 2)
    layer_fwd<TR, true>(m.p1t, h, m.c1, n, h, s.U, ph);
    __syncthreads();
    layer_fwd<1, false>(m.p2t, 4, m.c2, h, 4, ph, s.O);
    // log|psi| = 1/2 sum_d log pi_d: 16 partial sums per row
    {
        const int r = threadIdx.x % TR, part = threadIdx.x / TR;     // NT/TR = 16 parts
        float acc = 0.0f;
        for (int d = part; d < n; d += NT / TR) {
            const float a = s.A[d * TR + r];
            const float ls = log_sigmoid(s.U[d * TR + r] > 0.0f ? a : -a);
            acc += (m.n_up >= 0 && s.keep[d * TR + r] == 0.0f) ? 0.0f : ls;
        }
        s.red[part * TR + r] = acc;
    }
    __syncthreads();
    if (threadIdx.x < TR) {
        const int r = threadIdx.x;
        float acc = 0.0f;
#pragma unroll
        for (int p = 0; p < NT / TR; ++p) acc += s.red[p * TR + r];
        s.lp[r] = (m.n_up >= 0 && s.bad[r] != 0.0f) ? -INFINITY : 0.5f * acc;
        const int sel = (s.U[(n - 2) * TR + r] > 0.0f ? 2 : 0) + (s.U[(n - 1) * TR + r] > 0.0f ? 1 : 0);
        s.phi[r] = s.O[sel * TR + r];
    }
    __syncthreads();
}

__global__ void __launch_bounds__(NT) logpsi_simt_kernel(MadeDev m, const ulonglong2 *__restrict__ cfg, long long B,
                                                         float2 *__restrict__ out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Smem s = carve(smem_raw, m);
    for (long long blk = blockIdx.x; blk * TR < B; blk += gridDim.x) {
        if (threadIdx.x < TR) {
            const long long i = blk * TR + threadIdx.x;
            s.cfg[threadIdx.x] = (i < B) ? cfg[i] : make_ulonglong2(0, 0);
        }
        __syncthreads();
        forward_tile(m, s);
        if (threadIdx.x < TR) {
            const long long i = blk * TR + threadIdx.x;
            if (i < B) out[i] = make_float2(s.lp[threadIdx.x], s.phi[threadIdx.x]);
        }
        __syncthreads();
    }
}

// Sampler support: pi_hat(z_d = 1 | z_<d) for every buffer entry — the conditional of
// autoregressive position d with the Hamming-weight clamp of Eq. 14 (reading A13: with c spin-sigma bits set before d and
// m spin-sigma positions left, force 0 if c = n_sigma, force 1 if n_sigma - c = m).  Entries are 128-bit prefixes in qubit
// order with the undecided positions zero: by the MADE masks logit d does not depend on them.
__global__ void __launch_bounds__(NT) cond_kernel(MadeDev m, const ulonglong2 *__restrict__ cfg, long long E, int d,
                                                  int n_up, int n_down, float *__restrict__ p1_out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Smem s = carve(smem_raw, m);
    const int sig = __ldg(m.order + d) & 1;                      // spin of this position: even qubit = up, odd = down (Eq. 12)
    for (long long blk = blockIdx.x; blk * TR < E; blk += gridDim.x) {
        if (threadIdx.x < TR) {
            const long long i = blk * TR + threadIdx.x;
            s.cfg[threadIdx.x] = (i < E) ? cfg[i] : make_ulonglong2(0, 0);
        }
        __syncthreads();
        forward_tile(m, s);                                      // leaves the logits in s.A, the +-1 inputs in s.U
        if (threadIdx.x < TR) {
            const int r = threadIdx.x;
            const long long i = blk * TR + r;
            if (i < E) {
                float p1 = 1.0f / (1.0f + expf(-s.A[d * TR + r]));
                if (n_up >= 0) {
                    int c = 0, left = 0;
                    for (int k = 0; k < m.n; ++k) {
                        if ((__ldg(m.order + k) & 1) != sig) continue;
                        if (k < d) c += s.U[k * TR + r] > 0.0f; else ++left;
                    }
                    const int target = sig == 0 ? n_up : n_down;
                    if (c >= target) p1 = 0.0f;
                    if (target - c >= left) p1 = 1.0f;
                }
                p1_out[i] = p1;
            }
        }
        __syncthreads();
    }
}

// Fused (a2)-(a5) on CUDA cores.  CTA = TR samples x a contiguous range of unique-flip groups.
__global__ void __launch_bounds__(NT) eloc_simt_kernel(HamDev hm, MadeDev m, const ulonglong2 *__restrict__ x,
                                                       const float2 *__restrict__ base, long long B,
                                                       float2 *__restrict__ partial, int nsplit,
                                                       unsigned *__restrict__ max_ratio_bits) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Smem s = carve(smem_raw, m);
    const long long blk = blockIdx.x;
    const int split = blockIdx.y;
    const long long g_lo = hm.G * split / nsplit, g_hi = hm.G * (split + 1) / nsplit;
    const int r = threadIdx.x;
    const long long i = blk * TR + r;
    ulonglong2 xr = make_ulonglong2(0, 0);
    float2 b0 = make_float2(0.f, 0.f), E = make_float2(0.f, 0.f);
    float mr = 0.0f;
    if (r < TR && i < B) { xr = x[i]; b0 = base[i]; }
    for (long long g = g_lo; g < g_hi; ++g) {
        const ulonglong2 f = hm.flips[g];
        const bool diag = (f.x | f.y) == 0ull;
        if (!diag) {                                                   // uniform branch
            if (r < TR) s.cfg[r] = make_ulonglong2(xr.x ^ f.x, xr.y ^ f.y);     // (a2) x' = x xor f_g
            __syncthreads();
            forward_tile(m, s);                                        // (a4)
        }
        if (r < TR && i < B) {
            // (a3) S = sum_{t in g} c_t (-i)^{r_t} (-1)^{popcount(x & s_t)}
            float2 S = make_float2(0.f, 0.f);
            const uint32_t t1 = hm.offsets[g + 1];
            for (uint32_t t = hm.offsets[g]; t < t1; ++t) {
                const ulonglong2 zy = hm.zy[t];
                const float2 c = hm.cph[t];
                const float2 cs = nqs_signed(c, nqs_parity_sign(xr, zy));
                S.x += cs.x;
                S.y += cs.y;
            }
            // (a5) ratio = exp(dlog|psi|) * cis(dphi); E += S * ratio
            float rr = 1.0f, ri = 0.0f;
            if (!diag) {
                const float mag = expf(s.lp[r] - b0.x);
                float sn, cs;
                sincosf(s.phi[r] - b0.y, &sn, &cs);
                rr = mag * cs; ri = mag * sn;
                mr = fmaxf(mr, mag);
            } else {
                mr = fmaxf(mr, 1.0f);
            }
            E.x += S.x * rr - S.y * ri;
            E.y += S.x * ri + S.y * rr;
        }
    }
    if (r < TR && i < B) {
        partial[(size_t)split * B + i] = E;
        atomicMax(max_ratio_bits, __float_as_uint(mr));               // mr >= 0: uint order == float order
    }
}

__global__ void reduce_partials_kernel(const float2 *__restrict__ partial, int nsplit, long long B,
                                       float2 *__restrict__ eloc) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= B) return;
    float2 e = make_float2(0.f, 0.f);
    for (int s = 0; s < nsplit; ++s) {                                // fixed order: deterministic
        const float2 p = partial[(size_t)s * B + i];
        e.x += p.x; e.y += p.y;
    }
    eloc[i] = e;
}

// (a3) standalone.  CTA = 256 samples (two per thread: every staged term is loaded once for both) x a range of groups;
// term tiles are staged through shared memory with cp.async (double-buffered) and every staged term is reused by the
// 256 samples.  Per (sample, term) pair: 4 LOP3 (AND + XOR fold), 1 POPC, 1 shift, 2 LOP3 (sign), 2 FADD.
constexpr int CT_THREADS = 128;
constexpr int CT_SPT = 2;                 // samples per thread
constexpr int CT_ROWS = CT_THREADS * CT_SPT;
constexpr int CT_TILE = 512;

__device__ __forceinline__ void cp_async16(void *dst, const void *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src));
}
__device__ __forceinline__ void cp_async8(void *dst, const void *src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src));
}

__global__ void __launch_bounds__(CT_THREADS) contract_kernel(HamDev hm, const ulonglong2 *__restrict__ x, long long B,
                                                              long long g0, long long g1, int gsplit,
                                                              float2 *__restrict__ S_out) {
    __shared__ __align__(16) ulonglong2 s_zy[2][CT_TILE];
    __shared__ __align__(16) float2 s_c[2][CT_TILE];
    const long long ng = g1 - g0;
    const long long ga = g0 + ng * blockIdx.y / gsplit, gb = g0 + ng * (blockIdx.y + 1) / gsplit;
    if (ga >= gb) return;
    const long long i0 = (long long)blockIdx.x * CT_ROWS + threadIdx.x, i1 = i0 + CT_THREADS;     // coalesced stores per half
    const ulonglong2 xa = (i0 < B) ? x[i0] : make_ulonglong2(0, 0), xb = (i1 < B) ? x[i1] : make_ulonglong2(0, 0);
    const uint32_t t_begin = hm.offsets[ga], t_end = hm.offsets[gb];
    auto stage = [&](int buf, uint32_t t0) {
        for (int k = threadIdx.x; k < CT_TILE; k += CT_THREADS) {
            const uint32_t t = t0 + k;
            if (t < t_end) { cp_async16(&s_zy[buf][k], hm.zy + t); cp_async8(&s_c[buf][k], hm.cph + t); }
        }
        asm volatile("cp.async.commit_group;\n");
    };
    long long g = ga;
    uint32_t next_off = hm.offsets[g + 1];
    float2 Sa = make_float2(0.f, 0.f), Sb = Sa;
    int buf = 0;
    stage(0, t_begin);
    for (uint32_t t0 = t_begin; t0 < t_end; t0 += CT_TILE, buf ^= 1) {
        if (t0 + CT_TILE < t_end) { stage(buf ^ 1, t0 + CT_TILE); asm volatile("cp.async.wait_group 1;\n"); }
        else asm volatile("cp.async.wait_group 0;\n");
        __syncthreads();
        const int cnt = min((uint32_t)CT_TILE, t_end - t0);
        for (int k = 0; k < cnt; ++k) {
            while (t0 + k == next_off) {                               // uniform across the CTA
                float2 *row = S_out + (size_t)(g - g0) * B;
                if (i0 < B) row[i0] = Sa;
                if (i1 < B) row[i1] = Sb;
                Sa = Sb = make_float2(0.f, 0.f);
                ++g; next_off = hm.offsets[g + 1];
            }
            const ulonglong2 zy = s_zy[buf][k];
            const float2 c = s_c[buf][k];
            const float2 ca = nqs_signed(c, nqs_parity_sign(xa, zy)), cb = nqs_signed(c, nqs_parity_sign(xb, zy));
            Sa.x += ca.x; Sa.y += ca.y;
            Sb.x += cb.x; Sb.y += cb.y;
        }
        __syncthreads();
    }
    float2 *row = S_out + (size_t)(g - g0) * B;
    if (i0 < B) row[i0] = Sa;
    if (i1 < B) row[i1] = Sb;
}

// (a6) count-weighted statistics in fp64, one CTA, fixed summation order.
__global__ void __launch_bounds__(256) stats_kernel(const float2 *__restrict__ eloc, const long long *__restrict__ counts,
                                                    long long B, double *__restrict__ out4) {
    __shared__ double sh[4][256];
    double a0 = 0, a1 = 0, a2 = 0, a3 = 0;
    for (long long i = threadIdx.x; i < B; i += 256) {
        const double c = counts ? (double)counts[i] : 1.0;
        const float2 e = eloc[i];
        a0 += c; a1 += c * (double)e.x; a2 += c * (double)e.y;
        a3 += c * ((double)e.x * (double)e.x + (double)e.y * (double)e.y);
    }
    sh[0][threadIdx.x] = a0; sh[1][threadIdx.x] = a1; sh[2][threadIdx.x] = a2; sh[3][threadIdx.x] = a3;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s)
            for (int q = 0; q < 4; ++q) sh[q][threadIdx.x] += sh[q][threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x < 4) out4[threadIdx.x] += sh[threadIdx.x][0];
}

int num_sms() {
    static int sms = 0;
    if (!sms) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev); }
    return sms > 0 ? sms : 148;
}

}  // namespace

int launch_logpsi_simt(const MadeDev &m, const ulonglong2 *cfg, long long B, float2 *out, cudaStream_t st) {
    if (B <= 0) return NQS_OK;
    const size_t sb = smem_bytes(m);
    if (sb > 227 * 1024) return NQS_EUNSUPPORTED;
    if (cudaFuncSetAttribute(logpsi_simt_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb) != cudaSuccess) return NQS_ECUDA;
    const long long nblk = (B + TR - 1) / TR;
    const int grid = (int)(nblk < (long long)num_sms() * 8 ? nblk : (long long)num_sms() * 8);
    logpsi_simt_kernel<<<grid, NT, sb, st>>>(m, cfg, B, out);
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? NQS_OK : NQS_ECUDA;
}

int launch_cond_simt(const MadeDev &m, const ulonglong2 *cfg, long long E, int d, int n_up, int n_down, float *p1,
                     cudaStream_t st) {
    if (E <= 0) return NQS_OK;
    const size_t sb = smem_bytes(m);
    if (sb > 227 * 1024) return NQS_EUNSUPPORTED;
    if (cudaFuncSetAttribute(cond_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb) != cudaSuccess) return NQS_ECUDA;
    const long long nblk = (E + TR - 1) / TR;
    const int grid = (int)(nblk < (long long)num_sms() * 8 ? nblk : (long long)num_sms() * 8);
    cond_kernel<<<grid, NT, sb, st>>>(m, cfg, E, d, n_up, n_down, p1);
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? NQS_OK : NQS_ECUDA;
}

int launch_contract(const HamDev &hm, const ulonglong2 *x, long long B, long long g0, long long g1, float2 *S,
                    cudaStream_t st) {
    if (B <= 0 || g1 <= g0) return NQS_OK;
    const long long nb = (B + CT_ROWS - 1) / CT_ROWS;
    long long gs = (8ll * num_sms() + nb - 1) / nb;           // ~8 resident CTAs (32 warps) per SM: the term loop is latency-bound below that
    if (gs > g1 - g0) gs = g1 - g0;
    if (gs < 1) gs = 1;
    if (gs > 65535) gs = 65535;
    dim3 grid((unsigned)nb, (unsigned)gs);
    contract_kernel<<<grid, CT_THREADS, 0, st>>>(hm, x, B, g0, g1, (int)gs, S);
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? NQS_OK : NQS_ECUDA;
}

size_t eloc_simt_partial_bytes(long long B, int *nsplit, const HamDev &hm) {
    const long long nblk = (B + TR - 1) / TR;
    long long ns = (4ll * num_sms() + nblk - 1) / nblk;     // aim for >= 4 CTAs per SM
    if (ns > hm.G) ns = hm.G;
    if (ns < 1) ns = 1;
    if (ns > 4096) ns = 4096;
    *nsplit = (int)ns;
    return sizeof(float2) * (size_t)ns * (size_t)B;
}

int launch_eloc_simt(const HamDev &hm, const MadeDev &m, const ulonglong2 *x, const float2 *base, long long B,
                     float2 *eloc, float2 *partial, int nsplit, unsigned *max_ratio_bits, cudaStream_t st) {
    if (B <= 0) return NQS_OK;
    const size_t sb = smem_bytes(m);
    if (sb > 227 * 1024) return NQS_EUNSUPPORTED;
    if (cudaFuncSetAttribute(eloc_simt_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb) != cudaSuccess) return NQS_ECUDA;
    const long long nblk = (B + TR - 1) / TR;
    dim3 grid((unsigned)nblk, (unsigned)nsplit);
    eloc_simt_kernel<<<grid, NT, sb, st>>>(hm, m, x, base, B, partial, nsplit, max_ratio_bits);
    ++g_launch_count;
    if (cudaGetLastError() != cudaSuccess) return NQS_ECUDA;
    reduce_partials_kernel<<<(unsigned)((B + 255) / 256), 256, 0, st>>>(partial, nsplit, B, eloc);
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? NQS_OK : NQS_ECUDA;
}

int launch_stats(const float2 *eloc, const long long *counts, long long B, double *stats4, cudaStream_t st) {
    if (B <= 0) return NQS_OK;
    stats_kernel<<<1, 256, 0, st>>>(eloc, counts, B, stats4);
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? NQS_OK : NQS_ECUDA;
}
