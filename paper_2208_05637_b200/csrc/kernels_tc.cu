// Tensor-core path (NQS_PATH_TC): ONE persistent, warp-specialised sm_100a kernel that runs, per tile of
// 128 samples x 1 unique-flip group g,
//   (a2) x' = x xor f_g expanded to a +-1 fp16 operand tile in shared memory,
//   (a4) the MADE chain and the phase MLP as tcgen05 MMAs (fp16 operands, fp32 accumulation in TMEM):
//          phase hidden  P = relu(A0 . P1^T + c1)      SS-mode, 64-unit chunks -> smem -> D3p += P . P2^T
//          layer 1       A1 = relu(A0 . W1^T + b1)     SS-mode, 64-unit chunks -> TMEM (fp16, A operand)
//          layer 2       A2 = relu(A1 . W2^T + b2)     TS-mode (A from TMEM), all-zero 64x64 mask tiles skipped
//          layer 3       D3 += A2 . W3^T               SS-mode from the smem staging chunk
//   (a3) the Pauli contraction S[i,g] over the group's terms (popcount parity, (-i)^r folded into c),
//   (a5) ratio = exp(dlog|psi|) cis(dphi), E_i += S * ratio, kept in registers per sample.
// Weight tiles are pre-packed on the host into the exact shared-memory images (128B-swizzled / core-matrix
// K-major) in consumption order and streamed by the TMA engine (1-D bulk copies) through a ring of slots.
// PAPER.md:122-134 (Alg. 1), :84-96 (architecture, Eq. 8-10), :152-158 (Eq. 15-16).
#include <cstring>
#include <new>
#include <vector>
#include "nqs_internal.h"
#include "tc_ptx.cuh"

using namespace tc;

namespace {

constexpr int TILE_M = 128;
constexpr int CH = 64;                   // hidden-unit chunk (= D buffer columns = staging K-block)
constexpr int NTHREADS = 320;            // warp 0 producer, warp 1 MMA, warps 2..9 epilogue
constexpr int NEPI_WARPS = 8;
constexpr int MAX_NC = 8;                // hidden <= 512
// TMEM column map (512 columns allocated)
constexpr uint32_t TM_A1 = 0;            // fp16 A1[128][H] packed 2/column: H/2 <= 256 columns
constexpr uint32_t TM_D0 = 256, TM_D1 = 320;   // two 64-column fp32 accumulators
constexpr uint32_t TM_D3 = 384;          // layer-3 logits, KO <= 112 columns
constexpr uint32_t TM_D3P = 496;         // phase outputs, 16 columns

struct TcParams {
    int n, H, NC, KI, KO;
    const uint8_t *wimg;                 // packed weight tiles
    const uint2 *prog;                   // per-tile weight program: (byte offset, bytes), consumption order
    int nprog;
    uint32_t slot_bytes;
    int nslots;
    const float *bias;                   // [c1 H | b1 H | b2 H | b3 KO | c2 4] fp32
    uint8_t nzmask[MAX_NC];              // layer-2 non-empty 64x64 tiles: bit kb of nzmask[c']
    int mode;                            // 0 = logpsi, 1 = local energy
    const ulonglong2 *xpos;              // [B] configurations, bits in autoregressive POSITION order
    long long B;
    float2 *out;                         // mode 0: (log|psi|, phi) per row
    const ulonglong2 *fpos;              // [G] flips in position order
    const ulonglong2 *x;                 // [B] samples in qubit order (contraction parity)
    HamDev hm;
    const float2 *base;                  // [B] (log|psi|, phi) of the samples
    float *eloc;                         // [B][2], pre-initialised with the f = 0 group; atomically accumulated
    unsigned *max_ratio_bits;
    long long g_begin;                   // first group that needs a forward pass (1 if group 0 is f = 0)
};

struct SmemLayout {
    uint32_t a0, t0, t1, bias, bars, slots, total;
};

__host__ __device__ inline SmemLayout smem_layout(int KI, int H, int KO, uint32_t slot_bytes, int nslots) {
    SmemLayout L;
    uint32_t off = 0;
    L.a0 = off; off += (uint32_t)KI * 256;                      // [128][KI] fp16 core-matrix layout
    off = (off + 1023) & ~1023u;
    L.t0 = off; off += 16384;
    L.t1 = off; off += 16384;
    L.bias = off; off += (uint32_t)(3 * H + KO + 4) * 4;
    off = (off + 15) & ~15u;
    L.bars = off; off += 64 * 8;
    off = (off + 1023) & ~1023u;
    L.slots = off; off += slot_bytes * (uint32_t)nslots;
    L.total = off;
    return L;
}

// barrier indices inside the bars block
enum { BAR_A0 = 0, BAR_FINAL = 1, BAR_DFULL = 2, BAR_DEMPTY = 4, BAR_TFULL = 6, BAR_TEMPTY = 8, BAR_A1 = 10,
       BAR_WFULL = 18, BAR_WEMPTY = 40 };   // up to 22 slots

__device__ __forceinline__ uint32_t pack_relu_half2(float a, float b) {
    __half2 h = __floats2half2_rn(fmaxf(a, 0.0f), fmaxf(b, 0.0f));
    return *reinterpret_cast<uint32_t *>(&h);
}

__device__ __forceinline__ unsigned long long shr128(ulonglong2 a, int s) {      // low 64 bits of a >> s, 0 <= s < 128
    if (s == 0) return a.x;
    if (s < 64) return (a.x >> s) | (a.y << (64 - s));
    return a.y >> (s - 64);
}

__device__ __forceinline__ float log_sigmoid_fast(float t) {
    return fminf(t, 0.0f) - __logf(1.0f + __expf(-fabsf(t)));
}

__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&v)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                 : "r"(taddr));
}

__global__ void __launch_bounds__(NTHREADS, 1) eloc_tc_kernel(const TcParams p) {
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ uint32_t s_tmem_base;
    __shared__ float s_xchg[TILE_M][2];                 // ch=1 -> ch=0 hand-over of (partial log-sum, phi)
    const SmemLayout L = smem_layout(p.KI, p.H, p.KO, p.slot_bytes, p.nslots);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + L.bars);
    float *s_bias = reinterpret_cast<float *>(smem + L.bias);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int NC = p.NC, KI = p.KI, KO = p.KO, H = p.H;

    // ---- one-time setup ----
    if (threadIdx.x == 0) {
        mbar_init(&bars[BAR_A0], NEPI_WARPS);
        mbar_init(&bars[BAR_FINAL], 1);
        for (int b = 0; b < 2; ++b) {
            mbar_init(&bars[BAR_DFULL + b], 1);
            mbar_init(&bars[BAR_DEMPTY + b], NEPI_WARPS);
            mbar_init(&bars[BAR_TFULL + b], NEPI_WARPS);
            mbar_init(&bars[BAR_TEMPTY + b], 1);
        }
        for (int c = 0; c < MAX_NC; ++c) mbar_init(&bars[BAR_A1 + c], NEPI_WARPS);
        for (int s = 0; s < p.nslots; ++s) { mbar_init(&bars[BAR_WFULL + s], 1); mbar_init(&bars[BAR_WEMPTY + s], 1); }
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc(&s_tmem_base, 512);
    for (int i = threadIdx.x; i < 3 * H + KO + 4; i += NTHREADS) s_bias[i] = p.bias[i];
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = s_tmem_base;

    // ---- static tile schedule: contiguous range per CTA, sample-block major ----
    const long long nsb = (p.B + TILE_M - 1) / TILE_M;
    const long long Gnd = (p.mode == 1) ? (p.hm.G - p.g_begin) : 1;
    const long long ntiles = nsb * Gnd;
    const long long t_lo = ntiles * blockIdx.x / gridDim.x, t_hi = ntiles * (blockIdx.x + 1) / gridDim.x;

    if (warp == 0) {
        // =========================== weight-tile producer (TMA engine, 1-D bulk copies) ===========================
        if (lane == 0) {
            uint32_t it = 0;                                   // running weight-tile index
            for (long long t = t_lo; t < t_hi; ++t) {
                for (int e = 0; e < p.nprog; ++e, ++it) {
                    const uint2 pe = __ldg(&p.prog[e]);
                    const uint32_t slot = it % (uint32_t)p.nslots, rnd = it / (uint32_t)p.nslots;
                    mbar_wait(&bars[BAR_WEMPTY + slot], (rnd & 1) ^ 1);
                    mbar_arrive_expect_tx(&bars[BAR_WFULL + slot], pe.y);
                    bulk_g2s(smem + L.slots + slot * p.slot_bytes, p.wimg + pe.x, pe.y, &bars[BAR_WFULL + slot]);
                }
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer (one thread) ===========================
        if (lane == 0) {
            const uint32_t a0_addr = smem_u32(smem + L.a0);
            const uint32_t a0_sbo = (uint32_t)(KI / 8) * 128;
            const uint32_t t_addr[2] = {smem_u32(smem + L.t0), smem_u32(smem + L.t1)};
            const uint32_t slots_addr = smem_u32(smem + L.slots);
            const uint32_t id64 = idesc_f16(128, 64), idKO = idesc_f16(128, KO), id16 = idesc_f16(128, 16);
            const uint32_t dcol[2] = {TM_D0, TM_D1};
            uint32_t it = 0, jd = 0, jt_c = 0, tcount = 0;    // weight tiles, D chunks, staging chunks (consumer side), tiles
            auto wait_w = [&]() -> uint32_t {
                const uint32_t slot = it % (uint32_t)p.nslots, rnd = it / (uint32_t)p.nslots;
                mbar_wait(&bars[BAR_WFULL + slot], rnd & 1);
                tc_fence_after();
                return slot;
            };
            auto done_w = [&](uint32_t slot) { mma_commit(&bars[BAR_WEMPTY + slot]); ++it; };
            // input layer chunk (SS, A0 core-matrix layout x weight tile core-matrix layout) -> D buffer
            auto input_chunk = [&]() {
                const uint32_t b = jd & 1, rnd = jd >> 1;
                mbar_wait(&bars[BAR_DEMPTY + b], (rnd & 1) ^ 1);
                tc_fence_after();
                const uint32_t slot = wait_w();
                const uint32_t w_addr = slots_addr + slot * p.slot_bytes;
                for (int ks = 0; ks < KI / 16; ++ks)
                    mma_ss(tmem + dcol[b], desc_noswz(a0_addr + ks * 256, 128, a0_sbo),
                           desc_noswz(w_addr + ks * 256, 128, a0_sbo), id64, ks > 0);
                done_w(slot);
                mma_commit(&bars[BAR_DFULL + b]);
                ++jd;
            };
            // consume one staging chunk (64 hidden units, smem, 128B swizzle): dst += T . W^T, N = KO or 16
            auto staged_chunk = [&](uint32_t dst_col, uint32_t idesc, bool accumulate) {
                const uint32_t tb = jt_c & 1, rnd = jt_c >> 1;
                mbar_wait(&bars[BAR_TFULL + tb], rnd & 1);
                tc_fence_after();
                const uint32_t slot = wait_w();
                const uint32_t w_addr = slots_addr + slot * p.slot_bytes;
                for (int ks = 0; ks < 4; ++ks)
                    mma_ss(tmem + dst_col, desc_sw128(t_addr[tb] + ks * 32), desc_sw128(w_addr + ks * 32), idesc,
                           accumulate || ks > 0);
                done_w(slot);
                mma_commit(&bars[BAR_TEMPTY + tb]);
                ++jt_c;
            };
            for (long long t = t_lo; t < t_hi; ++t, ++tcount) {
                mbar_wait(&bars[BAR_A0], tcount & 1);
                tc_fence_after();
                // ---- phase MLP: hidden chunks, then (one chunk behind) P2 ----
                for (int c = 0; c < NC; ++c) {
                    input_chunk();
                    if (c >= 1) staged_chunk(TM_D3P, id16, c - 1 > 0);
                }
                staged_chunk(TM_D3P, id16, NC - 1 > 0);
                // ---- layer 1 -> A1 in TMEM (written by the epilogue warps) ----
                for (int c = 0; c < NC; ++c) input_chunk();
                // ---- layer 2 (TS) with layer 3 one chunk behind ----
                for (int c2 = 0; c2 < NC; ++c2) {
                    const uint32_t b = jd & 1, rnd = jd >> 1;
                    mbar_wait(&bars[BAR_DEMPTY + b], (rnd & 1) ^ 1);
                    tc_fence_after();
                    bool first = true;
                    for (int kb = 0; kb < NC; ++kb) {
                        if (!((p.nzmask[c2] >> kb) & 1)) continue;
                        mbar_wait(&bars[BAR_A1 + kb], tcount & 1);
                        tc_fence_after();
                        const uint32_t slot = wait_w();
                        const uint32_t w_addr = slots_addr + slot * p.slot_bytes;
                        for (int ks = 0; ks < 4; ++ks) {
                            mma_ts(tmem + dcol[b], tmem + TM_A1 + kb * 32 + ks * 8, desc_sw128(w_addr + ks * 32), id64,
                                   !first || ks > 0);
                        }
                        first = false;
                        done_w(slot);
                    }
                    mma_commit(&bars[BAR_DFULL + b]);
                    ++jd;
                    if (c2 >= 1) staged_chunk(TM_D3, idKO, c2 - 1 > 0);
                }
                staged_chunk(TM_D3, idKO, NC - 1 > 0);
                mma_commit(&bars[BAR_FINAL]);
            }
        }
    } else {
        // =========================== epilogue warps (256 threads) ===========================
        const int ew = warp - 2;
        const int q = warp & 3;                    // TMEM lane quadrant this warp may access
        const int ch = ew >> 2;                    // column half
        const int row = q * 32 + lane;
        const uint32_t lane_base = (uint32_t)(q * 32) << 16;
        const uint32_t dcol[2] = {TM_D0, TM_D1};
        uint8_t *a0 = smem + L.a0;
        uint8_t *tbuf[2] = {smem + L.t0, smem + L.t1};
        const uint32_t a0_sbo = (uint32_t)(KI / 8) * 128;
        const float *s_c1 = s_bias, *s_b1 = s_bias + H, *s_b2 = s_bias + 2 * H, *s_b3 = s_bias + 3 * H, *s_c2 = s_bias + 3 * H + KO;
        uint32_t jd = 0, jt_p = 0, tcount = 0;
        long long cur_sb = -1;
        ulonglong2 xp = make_ulonglong2(0, 0), xq = make_ulonglong2(0, 0);
        float2 b0 = make_float2(0.f, 0.f), E = make_float2(0.f, 0.f);
        float mr = (p.mode == 1 && p.hm.has_diag) ? 1.0f : 0.0f;     // the f = 0 group has ratio exactly 1
        long long my_i = -1;

        // one hidden chunk: TMEM accumulator -> +bias, ReLU, fp16 -> (to_tmem ? A1 in TMEM : staging smem)
        auto hidden_chunk = [&](const float *bias_vec, int c, bool to_tmem) {
            const uint32_t b = jd & 1, rnd = jd >> 1;
            mbar_wait(&bars[BAR_DFULL + b], rnd & 1);
            tc_fence_after();
            uint32_t v[32];
            tmem_ld32(tmem + lane_base + dcol[b] + ch * 32, v);
            tmem_wait_ld();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars[BAR_DEMPTY + b]);
            ++jd;
            uint32_t w[16];
            const float4 *bp = reinterpret_cast<const float4 *>(bias_vec + c * CH + ch * 32);
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const float4 bb = bp[j];
                w[2 * j] = pack_relu_half2(__uint_as_float(v[4 * j]) + bb.x, __uint_as_float(v[4 * j + 1]) + bb.y);
                w[2 * j + 1] = pack_relu_half2(__uint_as_float(v[4 * j + 2]) + bb.z, __uint_as_float(v[4 * j + 3]) + bb.w);
            }
            if (to_tmem) {
                tmem_st16(tmem + lane_base + TM_A1 + c * 32 + ch * 16, w);
                tmem_wait_st();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bars[BAR_A1 + c]);
            } else {
                const uint32_t tb = jt_p & 1, trnd = jt_p >> 1;
                mbar_wait(&bars[BAR_TEMPTY + tb], (trnd & 1) ^ 1);
                uint8_t *T = tbuf[tb];
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    *reinterpret_cast<uint4 *>(T + sw128_offset(row, ch * 32 + j * 8)) =
                        make_uint4(w[4 * j], w[4 * j + 1], w[4 * j + 2], w[4 * j + 3]);
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bars[BAR_TFULL + tb]);
                ++jt_p;
            }
        };

        for (long long t = t_lo; t < t_hi; ++t, ++tcount) {
            const long long sb = t / Gnd, g = p.g_begin + (t % Gnd);
            if (sb != cur_sb) {
                if (p.mode == 1 && ch == 0 && my_i >= 0 && my_i < p.B) {
                    atomicAdd(&p.eloc[2 * my_i], E.x);
                    atomicAdd(&p.eloc[2 * my_i + 1], E.y);
                }
                cur_sb = sb;
                my_i = sb * TILE_M + row;
                E = make_float2(0.f, 0.f);
                if (my_i < p.B) {
                    xp = p.xpos[my_i];
                    if (p.mode == 1) { xq = p.x[my_i]; b0 = p.base[my_i]; }
                } else {
                    xp = make_ulonglong2(0, 0); xq = xp; b0 = make_float2(0.f, 0.f);
                }
            }
            ulonglong2 zp = xp;
            if (p.mode == 1) { const ulonglong2 f = __ldg(&p.fpos[g]); zp.x ^= f.x; zp.y ^= f.y; }

            // ---- (a2) A0: +-1 fp16 tile, core-matrix K-major layout; this thread fills its half of the K chunks ----
            {
                const int nkc = KI / 8, kc0 = ch * ((nkc + 1) / 2), kc1 = ch ? nkc : (nkc + 1) / 2;
                for (int kc = kc0; kc < kc1; ++kc) {
                    const uint32_t bits = (uint32_t)(shr128(zp, kc * 8) & 0xFFull);
                    uint4 w;
                    w.x = 0xBC00BC00u ^ ((bits & 1u) << 15) ^ ((bits & 2u) << 30);
                    w.y = 0xBC00BC00u ^ ((bits & 4u) << 13) ^ ((bits & 8u) << 28);
                    w.z = 0xBC00BC00u ^ ((bits & 16u) << 11) ^ ((bits & 32u) << 26);
                    w.w = 0xBC00BC00u ^ ((bits & 64u) << 9) ^ ((bits & 128u) << 24);
                    *reinterpret_cast<uint4 *>(a0 + (row >> 3) * a0_sbo + kc * 128 + (row & 7) * 16) = w;
                }
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bars[BAR_A0]);
            }
            // ---- (a4) hidden chunks, in the MMA warp's order ----
            for (int c = 0; c < NC; ++c) hidden_chunk(s_c1, c, false);      // phase hidden -> staging -> P2
            for (int c = 0; c < NC; ++c) hidden_chunk(s_b1, c, true);       // layer 1 -> A1 (TMEM)
            for (int c = 0; c < NC; ++c) hidden_chunk(s_b2, c, false);      // layer 2 -> staging -> layer 3

            // ---- final epilogue: log|psi| = 1/2 sum_d log sigmoid(+-a_d), phi = o[2 z_{n-2} + z_{n-1}] ----
            mbar_wait(&bars[BAR_FINAL], tcount & 1);
            tc_fence_after();
            float part = 0.0f, phi = 0.0f;
            {
                const int half = KO / 2;                         // KO is a multiple of 16
                const int d0 = ch * half;
                for (int j = 0; j < half; j += 8) {
                    uint32_t v[8];
                    tmem_ld8(tmem + lane_base + TM_D3 + d0 + j, v);
                    tmem_wait_ld();
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        const int d = d0 + j + k;
                        if (d < p.n) {
                            const float a = __uint_as_float(v[k]) + s_b3[d];
                            const bool z = (shr128(zp, d) & 1ull) != 0;
                            part += log_sigmoid_fast(z ? a : -a);
                        }
                    }
                }
                if (ch == 1) {
                    uint32_t v[8];
                    tmem_ld8(tmem + lane_base + TM_D3P, v);
                    tmem_wait_ld();
                    const int sel = (int)((shr128(zp, p.n - 2) & 1ull) * 2 + (shr128(zp, p.n - 1) & 1ull));
                    const float o0 = __uint_as_float(v[0]) + s_c2[0], o1 = __uint_as_float(v[1]) + s_c2[1];
                    const float o2 = __uint_as_float(v[2]) + s_c2[2], o3 = __uint_as_float(v[3]) + s_c2[3];
                    phi = sel == 0 ? o0 : (sel == 1 ? o1 : (sel == 2 ? o2 : o3));
                    s_xchg[row][0] = part;
                    s_xchg[row][1] = phi;
                }
            }
            tc_fence_before();
            asm volatile("bar.sync 1, 256;\n" ::: "memory");                  // the 8 epilogue warps only
            if (ch == 0) {
                const float lp = 0.5f * (part + s_xchg[row][0]);
                phi = s_xchg[row][1];
                if (p.mode == 0) {
                    if (my_i < p.B) p.out[my_i] = make_float2(lp, phi);
                } else if (my_i < p.B) {
                    // (a3) S = sum_{t in g} c_t (-i)^{r_t} (-1)^{popcount(x & s_t)}
                    float2 S = make_float2(0.f, 0.f);
                    const uint32_t t1 = __ldg(&p.hm.offsets[g + 1]);
                    for (uint32_t tt = __ldg(&p.hm.offsets[g]); tt < t1; ++tt) {
                        const ulonglong2 zy = __ldg(&p.hm.zy[tt]);
                        const float2 c = __ldg(&p.hm.cph[tt]);
                        const bool neg = ((__popcll(xq.x & zy.x) + __popcll(xq.y & zy.y)) & 1) != 0;
                        S.x += neg ? -c.x : c.x;
                        S.y += neg ? -c.y : c.y;
                    }
                    // (a5)
                    const float mag = __expf(lp - b0.x);
                    float sn, cs;
                    __sincosf(phi - b0.y, &sn, &cs);
                    const float rr = mag * cs, ri = mag * sn;
                    mr = fmaxf(mr, mag);
                    E.x += S.x * rr - S.y * ri;
                    E.y += S.x * ri + S.y * rr;
                }
            }
            asm volatile("bar.sync 1, 256;\n" ::: "memory");                  // s_xchg reusable
        }
        if (p.mode == 1 && ch == 0 && my_i >= 0 && my_i < p.B) {
            atomicAdd(&p.eloc[2 * my_i], E.x);
            atomicAdd(&p.eloc[2 * my_i + 1], E.y);
            atomicMax(p.max_ratio_bits, __float_as_uint(mr));
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem, 512);
}

// position-ordered copy of 128-bit configurations: out bit d = in bit order[d]
__global__ void permute_bits_kernel(const ulonglong2 *__restrict__ in, long long N, const int32_t *__restrict__ order, int n,
                                    ulonglong2 *__restrict__ out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const ulonglong2 a = in[i];
    unsigned long long lo = 0, hi = 0;
    for (int d = 0; d < n; ++d) {
        const int qb = __ldg(order + d);
        const unsigned long long bit = ((qb < 64 ? a.x : a.y) >> (qb & 63)) & 1ull;
        if (d < 64) lo |= bit << d; else hi |= bit << (d - 64);
    }
    out[i] = make_ulonglong2(lo, hi);
}

// eloc[i] = S[i, group 0] when group 0 is the f = 0 group (psi ratio == 1), else 0.
__global__ void diag_init_kernel(HamDev hm, const ulonglong2 *__restrict__ x, long long B, float2 *__restrict__ eloc) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= B) return;
    float2 S = make_float2(0.f, 0.f);
    if (hm.has_diag) {
        const ulonglong2 xr = x[i];
        const uint32_t t1 = hm.offsets[1];
        for (uint32_t t = hm.offsets[0]; t < t1; ++t) {
            const ulonglong2 zy = __ldg(&hm.zy[t]);
            const float2 c = __ldg(&hm.cph[t]);
            const bool neg = ((__popcll(xr.x & zy.x) + __popcll(xr.y & zy.y)) & 1) != 0;
            S.x += neg ? -c.x : c.x;
            S.y += neg ? -c.y : c.y;
        }
    }
    eloc[i] = S;
}

}  // namespace

// ------------------------------------------------------------------------------------------------------------
struct TcPack {
    int KI = 0, KO = 0, NC = 0, nprog = 0, nslots = 0;
    uint32_t slot_bytes = 0;
    uint8_t nzmask[MAX_NC] = {0};
    void *d_wimg = nullptr, *d_prog = nullptr, *d_bias = nullptr;
    void *d_fpos = nullptr; size_t fpos_cap = 0; const void *fpos_for = nullptr; long long fpos_G = -1;
    void *d_xpos = nullptr; size_t xpos_cap = 0;
    SmemLayout L{};
    int sms = 148;
};

bool tc_supported(const nqs_made *M) {
    return M->L == 2 && M->h % CH == 0 && M->h >= 64 && M->h <= 512 && ((M->n + 15) / 16) * 16 <= 112;
}

static inline uint32_t noswz_offset(uint32_t r, uint32_t k, uint32_t KI) {
    return (r >> 3) * (KI / 8) * 128u + (k >> 3) * 128u + (r & 7u) * 16u + (k & 7u) * 2u;
}

int tc_pack_upload(const nqs_made *M) {
    if (M->tc) return NQS_OK;
    TcPack *P = new (std::nothrow) TcPack();
    if (!P) return NQS_ENOMEM;
    const int n = M->n, H = M->h, NC = H / CH;
    const int KI = ((n + 15) / 16) * 16, KO = KI;
    P->KI = KI; P->KO = KO; P->NC = NC;
    const uint32_t in_bytes = (uint32_t)CH * KI * 2, w2_bytes = CH * 128, w3_bytes = (uint32_t)KO * 128, p2_bytes = 16 * 128;
    uint32_t slot = in_bytes;
    if (w2_bytes > slot) slot = w2_bytes;
    if (w3_bytes > slot) slot = w3_bytes;
    slot = (slot + 1023) & ~1023u;
    P->slot_bytes = slot;
    std::vector<uint8_t> img;
    std::vector<uint2> prog;
    auto put = [&](uint32_t off, float v) { __half hv = __float2half_rn(v); memcpy(&img[off], &hv, 2); };
    auto new_tile = [&](uint32_t bytes) -> uint32_t {
        const uint32_t off = (uint32_t)img.size();
        img.resize(img.size() + ((bytes + 127) & ~127u), 0);
        prog.push_back(make_uint2(off, bytes));
        return off;
    };
    auto input_tile = [&](int c, bool phase) {
        const uint32_t off = new_tile(in_bytes);
        for (int r = 0; r < CH; ++r) {
            const int j = c * CH + r;
            for (int k = 0; k < KI; ++k) {
                float v = 0.f;
                if (phase) { if (k < n - 2) v = M->p1[(size_t)j * (n - 2) + k]; }
                else if (k < n) v = M->wm[0][(size_t)j * n + k];
                put(off + noswz_offset(r, k, KI), v);
            }
        }
    };
    auto p2_tile = [&](int c) {
        const uint32_t off = new_tile(p2_bytes);
        for (int o = 0; o < 4; ++o)
            for (int k = 0; k < CH; ++k) put(off + sw128_offset(o, k), M->p2[(size_t)o * H + c * CH + k]);
    };
    auto w3_tile = [&](int c) {
        const uint32_t off = new_tile(w3_bytes);
        for (int d = 0; d < n; ++d)
            for (int k = 0; k < CH; ++k) put(off + sw128_offset(d, k), M->wm[2][(size_t)d * H + c * CH + k]);
    };
    // layer-2 tile occupancy (exact: a tile is skipped only if every masked weight in it is 0)
    for (int c2 = 0; c2 < NC; ++c2) {
        uint8_t m = 0;
        for (int kb = 0; kb < NC; ++kb) {
            bool any = false;
            for (int r = 0; r < CH && !any; ++r)
                for (int k = 0; k < CH; ++k)
                    if (M->wm[1][(size_t)(c2 * CH + r) * H + kb * CH + k] != 0.0f) { any = true; break; }
            if (any) m |= (uint8_t)(1u << kb);
        }
        if (!m) m = 1;
        P->nzmask[c2] = m;
    }
    // consumption order (must mirror the MMA warp's program)
    for (int c = 0; c < NC; ++c) { input_tile(c, true); if (c >= 1) p2_tile(c - 1); }
    p2_tile(NC - 1);
    for (int c = 0; c < NC; ++c) input_tile(c, false);
    for (int c2 = 0; c2 < NC; ++c2) {
        for (int kb = 0; kb < NC; ++kb) {
            if (!((P->nzmask[c2] >> kb) & 1)) continue;
            const uint32_t off = new_tile(w2_bytes);
            for (int r = 0; r < CH; ++r)
                for (int k = 0; k < CH; ++k)
                    put(off + sw128_offset(r, k), M->wm[1][(size_t)(c2 * CH + r) * H + kb * CH + k]);
        }
        if (c2 >= 1) w3_tile(c2 - 1);
    }
    w3_tile(NC - 1);
    P->nprog = (int)prog.size();
    // biases: [c1 | b1 | b2 | b3 (KO) | c2]
    std::vector<float> bias((size_t)3 * H + KO + 4, 0.f);
    for (int j = 0; j < H; ++j) { bias[j] = M->c1[j]; bias[H + j] = M->bias[0][j]; bias[2 * H + j] = M->bias[1][j]; }
    for (int d = 0; d < n; ++d) bias[3 * H + d] = M->bias[2][d];
    for (int o = 0; o < 4; ++o) bias[3 * H + KO + o] = M->c2[o];
    // slots: as many as fit in 227 KB (max 22 barriers reserved)
    int ns = 22;
    while (ns > 2 && smem_layout(KI, H, KO, slot, ns).total > 227 * 1024 - 2048) --ns;
    P->nslots = ns;
    P->L = smem_layout(KI, H, KO, slot, ns);
    int dev = 0; cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&P->sms, cudaDevAttrMultiProcessorCount, dev);
    bool ok = cudaMalloc(&P->d_wimg, img.size()) == cudaSuccess && cudaMalloc(&P->d_prog, prog.size() * sizeof(uint2)) == cudaSuccess &&
              cudaMalloc(&P->d_bias, bias.size() * 4) == cudaSuccess;
    ok = ok && cudaMemcpy(P->d_wimg, img.data(), img.size(), cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(P->d_prog, prog.data(), prog.size() * sizeof(uint2), cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemcpy(P->d_bias, bias.data(), bias.size() * 4, cudaMemcpyHostToDevice) == cudaSuccess;
    ok = ok && cudaFuncSetAttribute(eloc_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P->L.total) == cudaSuccess;
    if (!ok) { cudaGetLastError(); cudaFree(P->d_wimg); cudaFree(P->d_prog); cudaFree(P->d_bias); delete P; return NQS_ECUDA; }
    M->tc = P;
    return NQS_OK;
}

void tc_pack_free(const nqs_made *M) {
    if (!M->tc) return;
    cudaFree(M->tc->d_wimg); cudaFree(M->tc->d_prog); cudaFree(M->tc->d_bias);
    if (M->tc->d_fpos) cudaFree(M->tc->d_fpos);
    if (M->tc->d_xpos) cudaFree(M->tc->d_xpos);
    delete M->tc;
    M->tc = nullptr;
}

static void fill_common(const nqs_made *M, TcParams &p) {
    const TcPack *P = M->tc;
    p.n = M->n; p.H = M->h; p.NC = P->NC; p.KI = P->KI; p.KO = P->KO;
    p.wimg = (const uint8_t *)P->d_wimg; p.prog = (const uint2 *)P->d_prog; p.nprog = P->nprog;
    p.slot_bytes = P->slot_bytes; p.nslots = P->nslots;
    p.bias = (const float *)P->d_bias;
    memcpy(p.nzmask, P->nzmask, MAX_NC);
}

static int ensure(void **buf, size_t *cap, size_t bytes) {
    if (*cap >= bytes) return NQS_OK;
    if (*buf) cudaFree(*buf);
    *buf = nullptr; *cap = 0;
    if (cudaMalloc(buf, bytes) != cudaSuccess) { cudaGetLastError(); return NQS_ENOMEM; }
    *cap = bytes;
    return NQS_OK;
}

static int permuted(const nqs_made *M, const ulonglong2 *in, long long N, ulonglong2 *out, cudaStream_t st) {
    permute_bits_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(in, N, M->dev.order, M->n, out);
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? NQS_OK : NQS_ECUDA;
}

int launch_logpsi_tc(const nqs_made *M, const ulonglong2 *cfg, long long B, float2 *out, cudaStream_t st) {
    if (B <= 0) return NQS_OK;
    TcPack *P = M->tc;
    if (!P) return NQS_EUNSUPPORTED;
    int rc = ensure(&P->d_xpos, &P->xpos_cap, sizeof(ulonglong2) * (size_t)B);
    if (rc) return rc;
    if ((rc = permuted(M, cfg, B, (ulonglong2 *)P->d_xpos, st))) return rc;
    TcParams p{};
    fill_common(M, p);
    p.mode = 0; p.xpos = (const ulonglong2 *)P->d_xpos; p.B = B; p.out = out;
    const long long ntiles = (B + TILE_M - 1) / TILE_M;
    const int grid = (int)(ntiles < P->sms ? ntiles : P->sms);
    eloc_tc_kernel<<<grid, NTHREADS, P->L.total, st>>>(p);
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? NQS_OK : NQS_ECUDA;
}

size_t eloc_tc_ws_bytes(long long, const HamDev &) { return 256; }

int launch_eloc_tc(const HamDev &hm, const nqs_made *M, const ulonglong2 *x, const float2 *base, long long B,
                   float2 *eloc, unsigned *max_ratio_bits, cudaStream_t st) {
    if (B <= 0) return NQS_OK;
    TcPack *P = M->tc;
    if (!P) return NQS_EUNSUPPORTED;
    int rc;
    // position-ordered flips, cached per Hamiltonian
    if (P->fpos_for != (const void *)hm.flips || P->fpos_G != hm.G) {
        if ((rc = ensure(&P->d_fpos, &P->fpos_cap, sizeof(ulonglong2) * (size_t)(hm.G ? hm.G : 1)))) return rc;
        if (hm.G > 0 && (rc = permuted(M, hm.flips, hm.G, (ulonglong2 *)P->d_fpos, st))) return rc;
        P->fpos_for = (const void *)hm.flips; P->fpos_G = hm.G;
    }
    if ((rc = ensure(&P->d_xpos, &P->xpos_cap, sizeof(ulonglong2) * (size_t)B))) return rc;
    if ((rc = permuted(M, x, B, (ulonglong2 *)P->d_xpos, st))) return rc;
    diag_init_kernel<<<(unsigned)((B + 255) / 256), 256, 0, st>>>(hm, x, B, eloc);
    ++g_launch_count;
    if (cudaGetLastError() != cudaSuccess) return NQS_ECUDA;
    TcParams p{};
    fill_common(M, p);
    p.mode = 1; p.xpos = (const ulonglong2 *)P->d_xpos; p.B = B; p.fpos = (const ulonglong2 *)P->d_fpos; p.x = x;
    p.hm = hm; p.base = base; p.eloc = (float *)eloc; p.max_ratio_bits = max_ratio_bits;
    p.g_begin = hm.has_diag ? 1 : 0;
    const long long nsb = (B + TILE_M - 1) / TILE_M;
    const long long ntiles = nsb * (hm.G - p.g_begin);
    if (ntiles > 0) {
        const int grid = (int)(ntiles < P->sms ? ntiles : P->sms);
        eloc_tc_kernel<<<grid, NTHREADS, P->L.total, st>>>(p);
        ++g_launch_count;
        if (cudaGetLastError() != cudaSuccess) return NQS_ECUDA;
    }
    return NQS_OK;
}
