// Internal structures of libnqs (not part of the ABI).
#pragma once
#include <cstdint>
#include <vector>
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include "../../include/nqs.h"

#define NQS_MAX_QUBITS 128
#define NQS_MAX_HIDDEN 1024

// ---- device views handed to kernels (plain pointers, no ownership) ------------------------------
struct HamDev {
    int n;
    long long K, G;
    const ulonglong2 *flips;     // [G] unique flip masks f_g (x = word 0, y = word 1), ascending
    const uint32_t   *offsets;   // [G+1] CSR into the term arrays
    const ulonglong2 *zy;        // [K] sign masks s_t
    const float2     *cph;       // [K] c_t * (-i)^{r_t}: (c,0), (0,-c), (-c,0), (0,c) for r mod 4 = 0..3
    int has_diag;                // 1 if flips[0] == 0 (group 0 connects x to itself: ratio == 1)
};

struct MadeDev {
    int n, h, L;
    int npad;                    // n rounded up to 4 (row stride of the transposed output layer)
    const int32_t *order;        // [n] position d -> qubit
    // SIMT pack: masked fp32 weights TRANSPOSED to [in][out] (out contiguous), position order
    const float *w1t;            // [n][h]
    const float *w2t;            // [h][h]   (NULL when L == 1)
    const float *w3t;            // [h][npad]
    const float *b1, *b2, *b3;   // [h], [h], [npad]
    const float *p1t;            // [n][h]   phase layer 1; rows n-2, n-1 are zero
    const float *p2t;            // [h][4]
    const float *c1, *c2;        // [h], [4]
    // exact work avoidance on the masked layers: output j of a layer needs inputs k < kend[j] only (1 + the last
    // non-zero masked weight of its row; for sorted degrees the masks are prefixes), the rest multiply exact zeros
    const int32_t *kend1, *kend2, *kend3;   // [h], [h] (NULL when L == 1), [n]
    // Hamming-weight constraint (Eq. 14; n_up < 0 = off): conditionals clamped to 0 / 1 contribute
    // log 1 = 0 to log|psi|; strings that violate Eq. 12 have psi = 0
    int n_up, n_down;
    unsigned long long spin_lo, spin_hi;   // bit d = 1 if autoregressive position d is a down spin (odd qubit, Eq. 12)
};

#ifdef __CUDACC__
// Sign bit of (-1)^{popcount(x & s)} (Eq. 16) as a float sign mask: 0x80000000 if the parity is odd.
// parity(a) ^ parity(b) = parity(a ^ b), so the four 32-bit words are AND-ed with the mask, XOR-folded (LOP3) and ONE
// popcount decides (POPC is a quarter-rate pipe; the straightforward form needs four).
__device__ __forceinline__ uint32_t nqs_parity_sign(ulonglong2 x, ulonglong2 s) {
    const unsigned long long f = (x.x & s.x) ^ (x.y & s.y);
    return (uint32_t)__popc((uint32_t)f ^ (uint32_t)(f >> 32)) << 31;
}
// c * (-1)^{parity}: flip the sign bits of (Re, Im)
__device__ __forceinline__ float2 nqs_signed(float2 c, uint32_t sign) {
    return make_float2(__uint_as_float(__float_as_uint(c.x) ^ sign), __uint_as_float(__float_as_uint(c.y) ^ sign));
}

// Positions whose conditional Eq. 14 clamps, for one configuration zp given in POSITION order (reading A13: at a
// position of spin s with c spin-s bits set before it and m spin-s positions left, forced to 0 if c = n_s, to 1 if
// n_s - c = m).  *valid = the string respects every clamp (equivalently satisfies Eq. 12).
__device__ __forceinline__ ulonglong2 nqs_forced_mask(ulonglong2 zp, int n, unsigned long long spin_lo, unsigned long long spin_hi,
                                                      int n_up, int n_down, bool *valid) {
    int cnt0 = 0, cnt1 = 0;
    int rem1 = __popcll(spin_lo) + __popcll(spin_hi), rem0 = n - rem1;
    unsigned long long f_lo = 0, f_hi = 0;
    bool ok = true;
    for (int d = 0; d < n; ++d) {
        const unsigned long long zw = d < 64 ? zp.x : zp.y, sw = d < 64 ? spin_lo : spin_hi;
        const int bit = (int)((zw >> (d & 63)) & 1ull), sig = (int)((sw >> (d & 63)) & 1ull);
        const int c = sig ? cnt1 : cnt0, left = sig ? rem1 : rem0, target = sig ? n_down : n_up;
        const bool f0 = c >= target, f1 = target - c >= left;
        if (f0 | f1) { if (d < 64) f_lo |= 1ull << d; else f_hi |= 1ull << (d - 64); }
        ok = ok && !(f0 && bit) && !(f1 && !bit);
        if (sig) { cnt1 += bit; --rem1; } else { cnt0 += bit; --rem0; }
    }
    *valid = ok;
    return make_ulonglong2(f_lo, f_hi);
}
#endif

// ---- handles ------------------------------------------------------------------------------------
struct nqs_ham {
    int n = 0;
    int64_t K = 0, G = 0;
    double sum_abs = 0.0;
    std::vector<uint64_t> flips, zy;      // [G][2], [K][2]
    std::vector<uint32_t> offsets;        // [G+1]
    std::vector<uint8_t>  ycount;         // [K]
    std::vector<float>    coef;           // [K]
    // device copy (lazy)
    mutable bool on_device = false;
    mutable int  device = -1;
    mutable void *d_flips = nullptr, *d_offsets = nullptr, *d_zy = nullptr, *d_cph = nullptr;
};

struct TcPack;   // tensor-core weight tiles of the CTA-pair kernel (kernels_tc.cu)
struct GradPack; // degree tables + workspace of the gradient path (kernels_grad.cu)

struct nqs_made {
    int n = 0, h = 0, L = 0, npad = 0;
    std::vector<int32_t> order;                 // [n]
    std::vector<int32_t> deg;                   // [L][h]
    std::vector<std::vector<float>> wm;         // masked weights, [out][in], position order (L+1)
    std::vector<std::vector<float>> bias;       // (L+1)
    std::vector<float> p1, p2, c1, c2;          // [h][n-2], [4][h], [h], [4]
    // device copies (lazy)
    mutable bool on_device = false;
    mutable int  device = -1;
    mutable std::vector<void *> d_allocs;
    mutable MadeDev dev{};
    mutable TcPack *tc = nullptr;
    mutable bool tc_failed = false;             // the tensor-core pack could not be built / uploaded: this handle runs on the fp32 path
    mutable GradPack *grad = nullptr;
    int n_up = -1, n_down = -1;                 // nqs_made_set_constraint
    // workspace (grown on demand, reused across calls)
    mutable void  *ws = nullptr;
    mutable size_t ws_bytes = 0;
    // staging buffers and stream of nqs_local_energy_host (grown on demand, reused across calls)
    mutable void *hx = nullptr, *hc = nullptr, *he = nullptr;
    mutable size_t h_rows = 0;
    mutable cudaStream_t h_stream = nullptr;
    // buffers of nqs_made_sample: one arena, grown on demand, reused across calls
    mutable void  *samp_ws = nullptr;
    mutable size_t samp_ws_bytes = 0;
    // timing of the chain kernel (nqs_last_chain_kernel_ms)
    mutable std::vector<cudaEvent_t> ev;        // pairs (start, stop)
    mutable int ev_used = 0;
};

// ---- shared helpers -----------------------------------------------------------------------------
extern long long g_launch_count;
int  nqs_check_device();                                        // NQS_OK / NQS_ECUDA / NQS_EARCH
int  nqs_ham_upload(const nqs_ham *ham);
int  nqs_made_upload(const nqs_made *made);
int  nqs_ws_reserve(const nqs_made *made, size_t bytes);
HamDev nqs_ham_dev(const nqs_ham *ham);

// kernels_simt.cu
int launch_logpsi_simt(const MadeDev &m, const ulonglong2 *cfg, long long B, float2 *out, cudaStream_t st);
int launch_contract(const HamDev &hm, const ulonglong2 *x, long long B, long long g0, long long g1,
                    float2 *S, cudaStream_t st);
int launch_eloc_simt(const HamDev &hm, const MadeDev &m, const ulonglong2 *x, const float2 *base, long long B,
                     float2 *eloc, float2 *partial, int nsplit, unsigned *max_ratio_bits, cudaStream_t st);
int launch_stats(const float2 *eloc, const long long *counts, long long B, double *stats4, cudaStream_t st);
size_t eloc_simt_partial_bytes(long long B, int *nsplit, const HamDev &hm);
int launch_cond_simt(const MadeDev &m, const ulonglong2 *cfg, long long E, int d, int n_up, int n_down, float *p1,
                     cudaStream_t st);

// kernels_tc.cu
bool tc_supported(const nqs_made *made);
int  tc_pack_upload(const nqs_made *made);
void tc_pack_free(const nqs_made *made);
int  launch_logpsi_tc(const nqs_made *made, const ulonglong2 *cfg, long long B, float2 *out, cudaStream_t st);
int  launch_eloc_tc(const HamDev &hm, const nqs_made *made, const ulonglong2 *x, const float2 *base, long long B,
                    float2 *eloc, unsigned *max_ratio_bits, cudaStream_t st);
size_t eloc_tc_ws_bytes(long long B, const HamDev &hm);
void tc_mma_counts(const nqs_made *made, long long *issued, long long *dense);   // K-steps per tile: issued / dense chain

// kernels_grad.cu
void grad_pack_free(const nqs_made *made);
