// Tensor-core path (NQS_PATH_TC): ONE persistent, warp-specialised sm_100a kernel that runs, per tile of
// 128 samples x 1 unique-flip group g,
//   (a2) x' = x xor f_g expanded to a +-1 fp16 operand tile A0 in shared memory (double-buffered),
//   (a4) the MADE chain and the phase MLP as tcgen05 MMAs (fp16 operands, fp32 accumulation in TMEM), in
//        64-unit hidden CHUNKS that ping-pong between two TMEM accumulators D[0] / D[1]:
//          layer 1   D = A0 . W1c^T        SS   -> epilogue: +b1, ReLU, fp16 -> A1 (TMEM, A operand of layer 2)
//          phase     D = A0 . P1c^T        SS   -> epilogue: +c1, ReLU, fp16 IN PLACE -> D3 += D . P2c^T   (TS)
//          layer 2   D = A1 . W2c^T        TS   -> epilogue: +b2, ReLU, fp16 IN PLACE -> D3 += D . W3c^T   (TS)
//        all-zero 64x16 blocks of the masked weights are never issued (exact: they contribute 0),
//   (a3) the Pauli contraction S[i,g] over the group's terms (popcount parity, (-i)^r folded into c),
//   (a5) ratio = exp(dlog|psi|) cis(dphi), E_i += S * ratio, kept in registers per sample.
// Warp roles (14 warps): 0 = weight producers (a few lanes issue TMA 1-D bulk copies into a ring of large smem slots;
// never more lanes than slots), 1 = MMA issuer (ONE elect.sync thread runs the fixed per-tile schedule; ring hand-over
// bits, K-step counts and k-block lists come from a host-built table in kernel-parameter space), 2-5 / 6-9 = two
// chunk-epilogue groups (one per accumulator), 10-13 = tile warps (build A0 of the NEXT tile, contraction, then the final
// epilogue of the current one).  The weight tiles are pre-packed on the host into the exact shared-memory images
// (128B-swizzled / core-matrix K-major) in consumption order.  What was measured and why the design is what it is:
// DESIGN.md sections 6-7.
// PAPER.md:122-134 (Alg. 1), :84-96 (architecture, Eq. 8-10), :152-158 (Eq. 15-16).
#include <cstring>
#include <new>
#include <vector>
#include "nqs_internal.h"
#include "tc_ptx.cuh"

using namespace tc;

namespace {

constexpr int TILE_M = 128;
constexpr int CH = 64;                   // hidden-unit chunk = accumulator columns
constexpr int NTHREADS = 448;
constexpr int MAX_NC = 8;                // hidden <= 512
constexpr int MAX_SLOTS = 16;
constexpr int NPROD = 4;                 // producer lanes (bulk-copy issuers)

// barrier ids
enum { BAR_A0FULL = 0, BAR_DFULL = 2, BAR_DFREE = 4, BAR_INPL = 6, BAR_D3FULL = 8, BAR_D3EMPTY = 9,
       BAR_WFULL = 10, BAR_WEMPTY = 10 + MAX_SLOTS, BAR_COUNT = 10 + 2 * MAX_SLOTS };

// Streamed weight sub-tiles are described by one 32-bit word each, in consumption order (kernel parameter
// space -> uniform loads): offset inside the ring slot, ring hand-over flags and one small per-tile number.
constexpr int MAX_SUB = 4 * MAX_NC + MAX_NC * MAX_NC;        // W1 + P1 + W2 blocks + W3
constexpr uint32_t SUB_OFF_MASK = 0x1FFFu;                   // [0:13)  byte offset inside the slot / 16 (slots <= 128 KB)
constexpr uint32_t SUB_NEW = 1u << 13;                       // first sub-tile of a ring fill: wait for the fill
constexpr uint32_t SUB_END = 1u << 14;                       // last sub-tile of a ring fill: release the slot
constexpr int SUB_AUX_SHIFT = 16;                            // [16:24) input chunks: K-steps to issue; W2: k-block; W3: n_lo / 16

struct ChunkOp { uint16_t bias_off; uint16_t dst_col; uint32_t kind; };   // kind 0: -> A1 at dst_col; 1: in place

struct SmemLayout { uint32_t a0, a0_bytes, res, bias, prog, chunks, bars, slots, total; };

__host__ __device__ inline SmemLayout smem_layout(int KI, int H, int KO, int NC, uint32_t slot_bytes, int nslots) {
    SmemLayout L;
    uint32_t off = 0;
    L.a0_bytes = (uint32_t)TILE_M * KI * 2;                      // [128][KI] fp16 core-matrix layout
    L.a0 = off; off += 2 * L.a0_bytes;
    off = (off + 1023) & ~1023u;
    L.res = off; off += (uint32_t)NC * 2048;                     // resident P2 tiles (16 rows x 64 K, 128B swizzle)
    L.bias = off; off += (uint32_t)(3 * H + KO + 4) * 4;
    off = (off + 15) & ~15u;
    L.prog = off;
    L.chunks = off; off += 3 * MAX_NC * (uint32_t)sizeof(ChunkOp);
    L.bars = off; off += BAR_COUNT * 8;
    off = (off + 1023) & ~1023u;
    L.slots = off; off += slot_bytes * (uint32_t)nslots;
    L.total = off;
    return L;
}

struct TcParams {
    int n, H, NC, KI, KO;
    uint32_t tm_d, tm_d3;                // TMEM columns: A1 at 0, D[0] at tm_d, D[1] at tm_d + 64, D3 at tm_d3
    const uint8_t *wimg;                 // packed streamed weight tiles
    const uint2 *fills;                  // per-tile ring fills: (byte offset, bytes), consumption order
    int nfills;
    uint32_t sub[MAX_SUB + 1];           // per-tile streamed sub-tiles (see SUB_*); one pad word (read-ahead)
    uint8_t nblk[MAX_NC];                // layer-2 k-blocks issued per output chunk
    const ChunkOp *chunks; int nchunks;  // per-tile accumulator chunks, in MMA order
    const uint8_t *resimg; uint32_t res_bytes;   // resident P2 tiles
    uint32_t slot_bytes; int nslots;
    const float *bias;                   // [c1 H | b1 H | b2 H | b3 KO | c2 4] fp32
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

__device__ __forceinline__ unsigned long long shr128(ulonglong2 a, int s) {      // low 64 bits of a >> s, 0 <= s < 128
    if (s == 0) return a.x;
    if (s < 64) return (a.x >> s) | (a.y << (64 - s));
    return a.y >> (s - 64);
}

__global__ void __launch_bounds__(NTHREADS, 1) eloc_tc_kernel(const __grid_constant__ TcParams p) {
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ uint32_t s_tmem_base;
    const SmemLayout L = smem_layout(p.KI, p.H, p.KO, p.NC, p.slot_bytes, p.nslots);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + L.bars);
    float *s_bias = reinterpret_cast<float *>(smem + L.bias);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int KI = p.KI, KO = p.KO, H = p.H;

    // ---- one-time setup ----
    if (threadIdx.x == 0) {
        mbar_init(&bars[BAR_A0FULL], 4); mbar_init(&bars[BAR_A0FULL + 1], 4);
        for (int b = 0; b < 2; ++b) {
            mbar_init(&bars[BAR_DFULL + b], 1);
            mbar_init(&bars[BAR_DFREE + b], 4);
            mbar_init(&bars[BAR_INPL + b], 4);
        }
        mbar_init(&bars[BAR_D3FULL], 1);
        mbar_init(&bars[BAR_D3EMPTY], 4);
        for (int s = 0; s < p.nslots; ++s) { mbar_init(&bars[BAR_WFULL + s], 1); mbar_init(&bars[BAR_WEMPTY + s], 1); }
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc(&s_tmem_base, 512);
    for (int i = threadIdx.x; i < 3 * H + KO + 4; i += NTHREADS) s_bias[i] = p.bias[i];
    for (int i = threadIdx.x; i < p.nchunks * (int)(sizeof(ChunkOp) / 8); i += NTHREADS)
        reinterpret_cast<uint2 *>(smem + L.chunks)[i] = reinterpret_cast<const uint2 *>(p.chunks)[i];
    for (int i = threadIdx.x; i < (int)(p.res_bytes / 16); i += NTHREADS)
        reinterpret_cast<uint4 *>(smem + L.res)[i] = reinterpret_cast<const uint4 *>(p.resimg)[i];
    fence_proxy_async();                                  // resident tiles are read by the tensor core (async proxy)
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
        // =========================== weight producers (TMA engine, 1-D bulk copies) ===========================
        // One thread sustains about one ring fill per ~700 cycles (measured: the rate does not depend on the fill
        // size), so NPROD lanes share the fills round-robin; fill q always lands in slot q % nslots.
        // Never more lanes than slots: a lane that runs two uses of a slot ahead of the consumer would see the
        // parity of an older phase and overwrite live data (parity waits alias after two phases).
        const uint32_t nprod = (uint32_t)(p.nslots < NPROD ? p.nslots : NPROD);
        if ((uint32_t)lane < nprod) {
            const long long total = (t_hi - t_lo) * (long long)p.nfills;
            uint32_t e = (uint32_t)lane % (uint32_t)p.nfills, slot = (uint32_t)lane % (uint32_t)p.nslots;
            uint32_t par = 1u ^ (((uint32_t)lane / (uint32_t)p.nslots) & 1u);   // a fresh barrier passes a parity-1 wait
            for (long long q = lane; q < total; q += nprod) {
                const uint2 pe = __ldg(&p.fills[e]);
                mbar_wait(&bars[BAR_WEMPTY + slot], par);
                mbar_arrive_expect_tx(&bars[BAR_WFULL + slot], pe.y);
                bulk_g2s(smem + L.slots + slot * p.slot_bytes, p.wimg + pe.x, pe.y, &bars[BAR_WFULL + slot]);
                e += nprod; while (e >= (uint32_t)p.nfills) e -= (uint32_t)p.nfills;
                slot += nprod; while (slot >= (uint32_t)p.nslots) { slot -= (uint32_t)p.nslots; par ^= 1u; }
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer: ONE elected thread ===========================
        // Inside an elect.sync region ptxas knows a single thread is active and moves operands to uniform registers
        // with plain R2UR; under `lane == 0` (or lane-predicated issue in a convergent warp) it emits a waterfall loop
        // (ELECT / R2UR.BROADCAST / BRA.U.ANY, ~12 instructions) around every tcgen05.mma.
        // The per-tile schedule is fixed code (stage A: layer 1 -> A1; stage P: phase hidden, in place, P2 one chunk
        // behind; stage C: layer 2 from A1, in place, W3 one chunk behind); only the ring hand-over bits, the K-step
        // counts and the k-block lists come from the parameter table.  Barrier parities live in the bits of `ph`.
        if (elect_one()) {
            const uint32_t issue = 1u;
            const uint32_t smem_base = smem_u32(smem);
            const uint32_t bars_addr = smem_base + L.bars;
            const uint32_t a0_lo0 = (smem_base + L.a0) >> 4, a0_step = L.a0_bytes >> 4;
            const uint32_t slots_lo = (smem_base + L.slots) >> 4, slot_step = p.slot_bytes >> 4, res_lo = (smem_base + L.res) >> 4;
            // descriptor words: lo = addr/16 | (lbo/16) << 16, hi = sbo/16 | version 1 << 14 | layout << 29
            const uint32_t lo_noswz = (128u >> 4) << 16, hi_noswz = (((uint32_t)(KI / 8) * 128u) >> 4) | (1u << 14);
            const uint32_t lo_sw128 = (16u >> 4) << 16, hi_sw128 = (1024u >> 4) | (1u << 14) | (2u << 29);
            const uint32_t id64 = idesc_f16(128, 64), id16 = idesc_f16(128, 16), id0 = idesc_f16(128, 0);
            const uint32_t NC = (uint32_t)p.NC, nslots = (uint32_t)p.nslots;
            const uint32_t tm_d = tmem + p.tm_d, tm_d3 = tmem + p.tm_d3, tm_ph = tm_d3 + (uint32_t)KO - 16;
            uint32_t ph = 0, slot = 0, wpar = 0, slot_lo = slots_lo, tcount = 0;
#define BAR_ADDR(id) (bars_addr + (uint32_t)(id) * 8u)
#define WAIT_BAR(id) do { mbar_spin(BAR_ADDR(id), (ph >> (id)) & 1u); ph ^= 1u << (id); tc_fence_after(); } while (0)
#define SLOT_ACQUIRE(w) do { if ((w) & SUB_NEW) { mbar_spin(BAR_ADDR(BAR_WFULL + slot), wpar); tc_fence_after(); } } while (0)
#define SLOT_RELEASE(w) do { if ((w) & SUB_END) { mma_commit_addr_if(issue, BAR_ADDR(BAR_WEMPTY + slot)); slot_lo += slot_step; \
                             if (++slot == nslots) { slot = 0; wpar ^= 1u; slot_lo = slots_lo; } } } while (0)
            // input-layer chunk (SS): D[b] = A0 . Wc^T over the first nk K-steps (a prefix: masked columns are the high ones)
            auto input_chunk = [&](uint32_t w, uint32_t a0_lo, uint32_t b) {
                SLOT_ACQUIRE(w);
                const uint32_t nk = (w >> SUB_AUX_SHIFT) & 0xFFu, d = tm_d + b * CH;
                const uint32_t a_lo = a0_lo | lo_noswz, b_lo = (slot_lo + (w & SUB_OFF_MASK)) | lo_noswz;
                mma_ss2(issue, d, a_lo, hi_noswz, b_lo, hi_noswz, id64, 0u);
                // nested so that the common exit is ONE taken branch (KI <= 128 -> at most 8 K-steps)
#define KSTEP(k) mma_ss2(issue, d, a_lo + 16u * (k), hi_noswz, b_lo + 16u * (k), hi_noswz, id64, 1u)
                if (nk > 1) { KSTEP(1); if (nk > 2) { KSTEP(2); if (nk > 3) { KSTEP(3); if (nk > 4) { KSTEP(4);
                if (nk > 5) { KSTEP(5); if (nk > 6) { KSTEP(6); if (nk > 7) { KSTEP(7); } } } } } } }
#undef KSTEP
                SLOT_RELEASE(w);
                mma_commit_addr_if(issue, BAR_ADDR(BAR_DFULL + b));
            };
            // consumer of the in-place fp16 chunk in D[b]: dst += D[b] . B^T, 4 K-steps of 16
            auto consume = [&](uint32_t b, uint32_t b_lo, uint32_t dst, uint32_t idesc) {
                const uint32_t a_t = tm_d + b * CH;
                b_lo |= lo_sw128;
#pragma unroll
                for (uint32_t ks = 0; ks < 4; ++ks) mma_ts2(issue, dst, a_t + 8 * ks, b_lo + 2 * ks, hi_sw128, idesc, 1u);
            };
            auto consume_phase = [&](uint32_t c, uint32_t b) {                  // P2 tile c is resident
                WAIT_BAR(BAR_INPL + b);
                if (c == 0) WAIT_BAR(BAR_D3EMPTY);                               // first write into D3 of this tile
                consume(b, res_lo + c * (2048u >> 4), tm_ph, id16);
            };
            auto consume_w3 = [&](uint32_t w, uint32_t b, bool last) {          // streamed layer-3 tile
                WAIT_BAR(BAR_INPL + b);
                SLOT_ACQUIRE(w);
                const uint32_t nlo = ((w >> SUB_AUX_SHIFT) & 0xFFu) * 16;       // output rows below n_lo receive exactly 0
                consume(b, slot_lo + (w & SUB_OFF_MASK) + (nlo / 8) * 64, tm_d3 + nlo, id0 | ((((uint32_t)KO - nlo) >> 3) << 17));
                SLOT_RELEASE(w);
                if (last) mma_commit_addr_if(issue, BAR_ADDR(BAR_D3FULL));
            };
            auto l2_chunk = [&](uint32_t c2, uint32_t b, uint32_t &si) {        // D[b] = A1 . W2[c2]^T over the listed k-blocks
                const uint32_t nb = p.nblk[c2], d = tm_d + b * CH;
                uint32_t w = p.sub[si];
#pragma unroll 1
                for (uint32_t j = 0; j < nb; ++j) {
                    const uint32_t wn = p.sub[si + 1];                           // next word early: hides the constant-load latency
                    ++si;
                    SLOT_ACQUIRE(w);
                    const uint32_t a_t = tmem + ((w >> SUB_AUX_SHIFT) & 0xFFu) * (CH / 2);
                    const uint32_t b_lo = (slot_lo + (w & SUB_OFF_MASK)) | lo_sw128;
                    mma_ts2(issue, d, a_t, b_lo, hi_sw128, id64, j);
                    mma_ts2(issue, d, a_t + 8, b_lo + 2, hi_sw128, id64, 1u);
                    mma_ts2(issue, d, a_t + 16, b_lo + 4, hi_sw128, id64, 1u);
                    mma_ts2(issue, d, a_t + 24, b_lo + 6, hi_sw128, id64, 1u);
                    SLOT_RELEASE(w);
                    w = wn;
                }
                mma_commit_addr_if(issue, BAR_ADDR(BAR_DFULL + b));
            };
            for (long long t = t_lo; t < t_hi; ++t, ++tcount) {
                const uint32_t a0_lo = a0_lo0 + (tcount & 1u) * a0_step;
                uint32_t si = 0;
                // ---- stage A: layer 1, epilogue -> A1 (frees the accumulator) ----
                WAIT_BAR(BAR_A0FULL + (tcount & 1u));
                for (uint32_t c = 0; c < NC; c += 2) {
                    if (c >= 2) WAIT_BAR(BAR_DFREE + 0);
                    input_chunk(p.sub[si++], a0_lo, 0);
                    if (c >= 2) WAIT_BAR(BAR_DFREE + 1);
                    input_chunk(p.sub[si++], a0_lo, 1);
                }
                // ---- stage P: phase hidden layer, in place; its consumer runs one chunk behind ----
                for (uint32_t c = 0; c < NC; c += 2) {
                    if (c == 0) WAIT_BAR(BAR_DFREE + 0);      // last stage-A chunk of group 0 (=> all of its A1 is written)
                    input_chunk(p.sub[si++], a0_lo, 0);
                    if (c >= 2) consume_phase(c - 1, 1);
                    if (c == 0) WAIT_BAR(BAR_DFREE + 1);
                    input_chunk(p.sub[si++], a0_lo, 1);
                    consume_phase(c, 0);
                }
                // ---- stage C: layer 2 from A1 (TS), in place; consumers (P2 of the last phase chunk, then W3) one behind ----
                for (uint32_t c2 = 0; c2 < NC; c2 += 2) {
                    l2_chunk(c2, 0, si);
                    if (c2 == 0) consume_phase(NC - 1, 1);
                    else consume_w3(p.sub[si++], 1, false);
                    l2_chunk(c2 + 1, 1, si);
                    consume_w3(p.sub[si++], 0, false);
                }
                consume_w3(p.sub[si++], 1, true);
            }
#undef BAR_ADDR
#undef WAIT_BAR
#undef SLOT_ACQUIRE
#undef SLOT_RELEASE
        }
        __syncwarp();
    } else if (warp < 10) {
        // =========================== chunk epilogue groups: group g owns accumulator D[g] ===========================
        const int grp = (warp - 2) >> 2;
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;     // TMEM lane quadrant of this warp
        const uint32_t d_addr = tmem + lane_base + p.tm_d + (uint32_t)grp * CH;
        const ChunkOp *chunks = reinterpret_cast<const ChunkOp *>(smem + L.chunks);
        uint32_t uses = 0;
        for (long long t = t_lo; t < t_hi; ++t) {
            for (int j = grp; j < p.nchunks; j += 2, ++uses) {
                const ChunkOp co = chunks[j];
                mbar_wait(&bars[BAR_DFULL + grp], uses & 1u);
                tc_fence_after();
                uint32_t v[64];
                tmem_ld32p(d_addr, v);
                tmem_ld32p(d_addr + 32, v + 32);
                tmem_wait_ld();
                const float4 *bp = reinterpret_cast<const float4 *>(s_bias + co.bias_off);
                uint32_t w[32];
#pragma unroll
                for (int j4 = 0; j4 < 16; ++j4) {
                    const float4 bb = bp[j4];
                    w[2 * j4] = cvt_relu_f16x2(__uint_as_float(v[4 * j4]) + bb.x, __uint_as_float(v[4 * j4 + 1]) + bb.y);
                    w[2 * j4 + 1] = cvt_relu_f16x2(__uint_as_float(v[4 * j4 + 2]) + bb.z, __uint_as_float(v[4 * j4 + 3]) + bb.w);
                }
                const bool inplace = co.kind != 0;
                tmem_st32(inplace ? d_addr : (tmem + lane_base + co.dst_col), w);
                tmem_wait_st();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bars[(inplace ? BAR_INPL : BAR_DFREE) + grp]);
            }
        }
    } else {
        // =========================== tile warps: A0 of the next tile, final epilogue of the current ===========================
        const int q = warp & 3;
        const int row = q * 32 + lane;
        const uint32_t lane_base = (uint32_t)(q * 32) << 16;
        const uint32_t d3_addr = tmem + lane_base + p.tm_d3;
        const uint32_t a0_sbo = (uint32_t)(KI / 8) * 128;
        const float *s_b3 = s_bias + 3 * H, *s_c2 = s_bias + 3 * H + KO;
        const uint32_t zero16[16] = {0};

        struct RowState { long long sb, i; ulonglong2 xp, xq; float2 b0; };
        auto load_row = [&](long long sb, RowState &r) {
            r.sb = sb; r.i = sb * TILE_M + row;
            if (r.i < p.B) {
                r.xp = p.xpos[r.i];
                if (p.mode == 1) { r.xq = p.x[r.i]; r.b0 = p.base[r.i]; }
                else { r.xq = make_ulonglong2(0, 0); r.b0 = make_float2(0.f, 0.f); }
            } else { r.xp = make_ulonglong2(0, 0); r.xq = r.xp; r.b0 = make_float2(0.f, 0.f); }
        };
        // (a2) A0: +-1 fp16 tile, core-matrix K-major layout, one row per thread
        auto build_a0 = [&](uint32_t buf, ulonglong2 zp) {
            uint8_t *a0 = smem + L.a0 + buf * L.a0_bytes + (row >> 3) * a0_sbo + (row & 7) * 16;
            for (int kc = 0; kc < KI / 8; ++kc) {
                const uint32_t bits = (uint32_t)(shr128(zp, kc * 8) & 0xFFull);
                uint4 w;
                w.x = 0xBC00BC00u ^ ((bits & 1u) << 15) ^ ((bits & 2u) << 30);
                w.y = 0xBC00BC00u ^ ((bits & 4u) << 13) ^ ((bits & 8u) << 28);
                w.z = 0xBC00BC00u ^ ((bits & 16u) << 11) ^ ((bits & 32u) << 26);
                w.w = 0xBC00BC00u ^ ((bits & 64u) << 9) ^ ((bits & 128u) << 24);
                *reinterpret_cast<uint4 *>(a0 + kc * 128) = w;
            }
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars[BAR_A0FULL + buf]);
        };
        auto flip_of = [&](long long t) -> ulonglong2 {
            if (p.mode != 1) return make_ulonglong2(0, 0);
            return __ldg(&p.fpos[p.g_begin + (t % Gnd)]);
        };

        // D3 accumulates from zero (every MMA into it has accumulate = 1)
        for (int c = 0; c < KO; c += 16) tmem_st16(d3_addr + c, zero16);
        tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars[BAR_D3EMPTY]);

        RowState cur{}, nxt{};
        ulonglong2 zp = make_ulonglong2(0, 0), zp_n = zp;
        float2 E = make_float2(0.f, 0.f);
        float mr = (p.mode == 1 && p.hm.has_diag) ? 1.0f : 0.0f;     // the f = 0 group has ratio exactly 1
        uint32_t tcount = 0;
        if (t_lo < t_hi) {
            load_row(t_lo / Gnd, cur);
            const ulonglong2 f = flip_of(t_lo);
            zp = make_ulonglong2(cur.xp.x ^ f.x, cur.xp.y ^ f.y);
            build_a0(0, zp);
        }
        for (long long t = t_lo; t < t_hi; ++t, ++tcount) {
            const long long g = p.g_begin + (t % Gnd);
            // ---- operand tile of the NEXT tile (its buffer was last read by tile t-1, whose D3FULL we have seen) ----
            const bool has_next = t + 1 < t_hi;
            if (has_next) {
                const long long sbn = (t + 1) / Gnd;
                if (sbn != cur.sb) load_row(sbn, nxt); else nxt = cur;
                const ulonglong2 f = flip_of(t + 1);
                zp_n = make_ulonglong2(nxt.xp.x ^ f.x, nxt.xp.y ^ f.y);
                build_a0((tcount + 1) & 1u, zp_n);
            }
            // ---- (a3) S = sum_{t in g} c_t (-i)^{r_t} (-1)^{popcount(x & s_t)}: independent of the MMAs, done while they run ----
            float2 S = make_float2(0.f, 0.f);
            if (p.mode == 1 && cur.i < p.B) {
                const uint32_t t1 = __ldg(&p.hm.offsets[g + 1]);
                for (uint32_t tt = __ldg(&p.hm.offsets[g]); tt < t1; ++tt) {
                    const ulonglong2 zy = __ldg(&p.hm.zy[tt]);
                    const float2 c = __ldg(&p.hm.cph[tt]);
                    const bool neg = ((__popcll(cur.xq.x & zy.x) + __popcll(cur.xq.y & zy.y)) & 1) != 0;
                    S.x += neg ? -c.x : c.x;
                    S.y += neg ? -c.y : c.y;
                }
            }
            // ---- final epilogue: log|psi| = 1/2 sum_d log sigmoid(+-a_d), phi = o[2 z_{n-2} + z_{n-1}] ----
            mbar_wait(&bars[BAR_D3FULL], tcount & 1u);
            tc_fence_after();
            // sum_d log sigmoid(t_d) = sum_d min(t_d, 0) - ln prod_d (1 + exp(-|t_d|)): every factor is in (1, 2], so a
            // 16-term product cannot overflow and costs one LG2 per 16 conditionals; the 16 chains are independent (ILP).
            float msum = 0.0f, lg = 0.0f, phi = 0.0f;
            for (int c0 = 0; c0 < KO; c0 += 16) {
                uint32_t v[16];
                tmem_ld16p(d3_addr + c0, v);
                tmem_wait_ld();
                tmem_st16(d3_addr + c0, zero16);              // D3 restarts from zero for the next tile
                if (c0 + 16 >= KO) {
                    const int sel = (int)((shr128(zp, p.n - 2) & 1ull) * 2 + (shr128(zp, p.n - 1) & 1ull));
                    const float o0 = __uint_as_float(v[12]) + s_c2[0], o1 = __uint_as_float(v[13]) + s_c2[1];
                    const float o2 = __uint_as_float(v[14]) + s_c2[2], o3 = __uint_as_float(v[15]) + s_c2[3];
                    phi = sel == 0 ? o0 : (sel == 1 ? o1 : (sel == 2 ? o2 : o3));
                }
                const uint32_t zb = (uint32_t)shr128(zp, c0);
                const int nv = p.n - c0;                       // valid conditionals in this block (may be <= 0 or >= 16)
                const float4 *bp = reinterpret_cast<const float4 *>(s_b3 + c0);
                float prod0 = 1.0f, prod1 = 1.0f, m0 = 0.0f, m1 = 0.0f;
#pragma unroll
                for (int k4 = 0; k4 < 4; ++k4) {
                    const float4 bb = bp[k4];
                    const float bk[4] = {bb.x, bb.y, bb.z, bb.w};
#pragma unroll
                    for (int kk = 0; kk < 4; ++kk) {
                        const int k = 4 * k4 + kk;
                        const float a = __uint_as_float(v[k]) + bk[kk];
                        float t = ((zb >> k) & 1u) ? a : -a;
                        t = (k < nv) ? t : 1e30f;              // padding column: factor 1, min 0
                        const float e = ex2_ftz(fabsf(t) * -1.4426950408889634f);
                        if (k & 1) { prod1 *= 1.0f + e; m1 += fminf(t, 0.0f); }
                        else       { prod0 *= 1.0f + e; m0 += fminf(t, 0.0f); }
                    }
                }
                msum += m0 + m1;
                lg += lg2_ftz(prod0 * prod1);
            }
            const float part = msum - 0.6931471805599453f * lg;
            tmem_wait_st();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars[BAR_D3EMPTY]);
            const float lp = 0.5f * part;
            if (p.mode == 0) {
                if (cur.i < p.B) p.out[cur.i] = make_float2(lp, phi);
            } else if (cur.i < p.B) {
                // (a5)
                const float mag = __expf(lp - cur.b0.x);
                float sn, cs;
                __sincosf(phi - cur.b0.y, &sn, &cs);
                const float rr = mag * cs, ri = mag * sn;
                mr = fmaxf(mr, mag);
                E.x += S.x * rr - S.y * ri;
                E.y += S.x * ri + S.y * rr;
            }
            if (!has_next || nxt.sb != cur.sb) {
                if (p.mode == 1 && cur.i < p.B) {
                    atomicAdd(&p.eloc[2 * cur.i], E.x);
                    atomicAdd(&p.eloc[2 * cur.i + 1], E.y);
                }
                E = make_float2(0.f, 0.f);
            }
            cur = nxt; zp = zp_n;
        }
        if (p.mode == 1) atomicMax(p.max_ratio_bits, __float_as_uint(mr));
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
    int KI = 0, KO = 0, NC = 0, nsub = 0, nchunks = 0, nfills = 0, nslots = 0;
    uint32_t slot_bytes = 0, res_bytes = 0, tm_d = 0, tm_d3 = 0;
    void *d_wimg = nullptr, *d_fills = nullptr, *d_chunks = nullptr, *d_res = nullptr, *d_bias = nullptr;
    void *d_fpos = nullptr; size_t fpos_cap = 0;
    void *d_xpos = nullptr; size_t xpos_cap = 0;
    SmemLayout L{};
    uint32_t sub[MAX_SUB + 1] = {0};
    uint8_t nblk[MAX_NC] = {0};
    int sms = 148;
    long long mma_issued = 0, mma_dense = 0;                   // K-steps issued / K-steps of the dense chain, per tile
};

static inline int round16(int v) { return (v + 15) / 16 * 16; }

static bool tc_shape(const nqs_made *M, int *KI_, int *KO_, uint32_t *slot_, int *nslots_) {
    if (M->L != 2 || M->h % (2 * CH) != 0 || M->h < 2 * CH || M->h > CH * MAX_NC) return false;
    const int KI = round16(M->n), KO = round16(M->n + 4), NC = M->h / CH;
    if (KI > 128 || KO > 128 || M->h / 2 + 2 * CH + KO > 512) return false;
    uint32_t slot = (uint32_t)CH * KI * 2;                                  // input sub-tile (64 rows x KI)
    if ((uint32_t)CH * 128 > slot) slot = CH * 128;                          // layer-2 sub-tile (64 x 64)
    if ((uint32_t)KO * 128 > slot) slot = (uint32_t)KO * 128;                // layer-3 sub-tile (KO x 64)
    slot = ((2 * slot) + 1023) & ~1023u;                                     // at least two sub-tiles per fill
    if (slot < 81920u) slot = 81920u;                                        // few, large bulk copies (a thread sustains ~1 copy / 700 cycles)
    int ns = MAX_SLOTS;
    while (ns > 0 && smem_layout(KI, M->h, KO, NC, slot, ns).total > 227 * 1024 - 1024) --ns;
    if (ns < 2) return false;
    *KI_ = KI; *KO_ = KO; *slot_ = slot; *nslots_ = ns;
    return true;
}

bool tc_supported(const nqs_made *M) {
    int KI, KO, ns; uint32_t slot;
    return tc_shape(M, &KI, &KO, &slot, &ns);
}

static inline uint32_t noswz_offset(uint32_t r, uint32_t k, uint32_t KI) {
    return (r >> 3) * (KI / 8) * 128u + (k >> 3) * 128u + (r & 7u) * 16u + (k & 7u) * 2u;
}

int tc_pack_upload(const nqs_made *M) {
    if (M->tc) return NQS_OK;
    int KI, KO, ns; uint32_t slot;
    if (!tc_shape(M, &KI, &KO, &slot, &ns)) return NQS_EUNSUPPORTED;
    TcPack *P = new (std::nothrow) TcPack();
    if (!P) return NQS_ENOMEM;
    const int n = M->n, H = M->h, NC = H / CH;
    P->KI = KI; P->KO = KO; P->NC = NC; P->slot_bytes = slot; P->nslots = ns;
    P->tm_d = (uint32_t)H / 2; P->tm_d3 = (uint32_t)H / 2 + 2 * CH;
    P->L = smem_layout(KI, H, KO, NC, slot, ns);
    const uint32_t in_bytes = (uint32_t)CH * KI * 2, w2_bytes = CH * 128, w3_bytes = (uint32_t)KO * 128;

    std::vector<uint8_t> img, res((size_t)NC * 2048, 0);
    std::vector<uint2> fills;
    std::vector<uint32_t> sub;
    std::vector<ChunkOp> chunks;
    auto put = [](std::vector<uint8_t> &buf, uint32_t off, float v) { __half hv = __float2half_rn(v); memcpy(&buf[off], &hv, 2); };

    // ---- streamed sub-tiles are appended to the open ring fill (<= slot bytes, in consumption order) ----
    uint32_t fill_start = 0, fill_bytes = 0;
    auto close_fill = [&]() {
        if (fill_bytes == 0) return;
        fills.push_back(make_uint2(fill_start, fill_bytes));
        sub.back() |= SUB_END;
        fill_bytes = 0;
    };
    // reserve `bytes` of streamed image for the next sub-tile; pushes its table word, returns its image offset
    auto stream_alloc = [&](uint32_t bytes, uint32_t aux) -> uint32_t {
        if (fill_bytes + bytes > slot) close_fill();
        uint32_t w = (aux & 0xFFu) << SUB_AUX_SHIFT;
        if (fill_bytes == 0) { fill_start = (uint32_t)img.size(); w |= SUB_NEW; }
        w |= (fill_bytes >> 4) & SUB_OFF_MASK;
        const uint32_t base = fill_start + fill_bytes;
        img.resize(img.size() + bytes, 0);
        fill_bytes += bytes;
        sub.push_back(w);
        return base;
    };

    // input-layer chunk c (layer 1 or phase hidden): D = A0 . Wc^T.  Masked layer-1 columns are the high ones
    // (M1[j][d] = deg[j] >= d+1), so the K-steps to issue are a prefix.
    auto input_chunk = [&](int c, bool phase) {
        const uint32_t base = stream_alloc(in_bytes, 0);
        int nk = 1;                                             // the accumulator must be overwritten even if all zero
        for (int r = 0; r < CH; ++r) {
            const int j = c * CH + r;
            for (int k = 0; k < KI; ++k) {
                float v = 0.f;
                if (phase) { if (k < n - 2) v = M->p1[(size_t)j * (n - 2) + k]; }
                else if (k < n) v = M->wm[0][(size_t)j * n + k];
                put(img, base + noswz_offset(r, k, KI), v);
                if (v != 0.0f && k / 16 + 1 > nk) nk = k / 16 + 1;
            }
        }
        sub.back() |= (uint32_t)nk << SUB_AUX_SHIFT;
        P->mma_issued += nk; P->mma_dense += KI / 16;
        ChunkOp co{};
        co.bias_off = (uint16_t)((phase ? 0 : H) + c * CH);
        co.kind = phase ? 1 : 0;
        co.dst_col = (uint16_t)(c * (CH / 2));
        chunks.push_back(co);
    };
    // resident P2 tile of phase chunk c: rows 12..15 of a 16-row tile hold the 4 phase outputs
    auto phase_out_tile = [&](int c) {
        for (int o = 0; o < 4; ++o)
            for (int k = 0; k < CH; ++k) put(res, (uint32_t)c * 2048 + sw128_offset(12 + o, k), M->p2[(size_t)o * H + c * CH + k]);
        P->mma_issued += 4; P->mma_dense += 4;
    };
    // streamed layer-3 tile of hidden chunk c; output rows below the first nonzero one receive exactly 0 from this
    // chunk, so the MMA starts at a 16-row boundary n_lo (Mout[d][j] = d+1 > deg[j])
    auto w3_tile = [&](int c) {
        const uint32_t base = stream_alloc(w3_bytes, 0);
        int row_lo = KO;
        for (int d = 0; d < n; ++d)
            for (int k = 0; k < CH; ++k) {
                const float v = M->wm[2][(size_t)d * H + c * CH + k];
                put(img, base + sw128_offset(d, k), v);
                if (v != 0.0f && d < row_lo) row_lo = d;
            }
        const int n_lo = row_lo >= KO ? 0 : (row_lo / 16) * 16;
        sub.back() |= (uint32_t)(n_lo / 16) << SUB_AUX_SHIFT;
        P->mma_issued += 4; P->mma_dense += 4;
    };

    // ---- the per-tile schedule (must match the MMA issuer in eloc_tc_kernel) ----
    for (int c = 0; c < NC; ++c) input_chunk(c, false);                          // stage A: layer 1 -> A1
    for (int c = 0; c < NC; ++c) { input_chunk(c, true); phase_out_tile(c); }     // stage P: phase hidden, in place
    uint8_t nblk[MAX_NC] = {0};
    for (int c2 = 0; c2 < NC; ++c2) {                                             // stage C: layer 2 (TS), in place
        int nb = 0;
        for (int kb = 0; kb < NC; ++kb) {
            bool any = false;
            for (int r = 0; r < CH && !any; ++r)
                for (int k = 0; k < CH; ++k)
                    if (M->wm[1][(size_t)(c2 * CH + r) * H + kb * CH + k] != 0.0f) { any = true; break; }
            P->mma_dense += 4;
            if (!any && !(nb == 0 && kb == NC - 1)) continue;                     // exact: an all-zero block adds 0
            const uint32_t base = stream_alloc(w2_bytes, (uint32_t)kb);
            for (int r = 0; r < CH; ++r)
                for (int k = 0; k < CH; ++k)
                    put(img, base + sw128_offset(r, k), M->wm[1][(size_t)(c2 * CH + r) * H + kb * CH + k]);
            P->mma_issued += 4;
            ++nb;
        }
        nblk[c2] = (uint8_t)nb;
        ChunkOp co{};
        co.bias_off = (uint16_t)(2 * H + c2 * CH); co.kind = 1; co.dst_col = 0;
        chunks.push_back(co);
        if (c2 >= 1) w3_tile(c2 - 1);                                             // consumer of the previous layer-2 chunk
    }
    w3_tile(NC - 1);
    close_fill();
    P->nsub = (int)sub.size(); P->nchunks = (int)chunks.size(); P->nfills = (int)fills.size();
    P->res_bytes = (uint32_t)res.size();
    if (P->nsub > MAX_SUB || (P->nchunks & 1)) { delete P; return NQS_EUNSUPPORTED; }
    memcpy(P->sub, sub.data(), sub.size() * 4);
    memcpy(P->nblk, nblk, sizeof(nblk));

    // biases: [c1 | b1 | b2 | b3 (KO) | c2]
    std::vector<float> bias((size_t)3 * H + KO + 4, 0.f);
    for (int j = 0; j < H; ++j) { bias[j] = M->c1[j]; bias[H + j] = M->bias[0][j]; bias[2 * H + j] = M->bias[1][j]; }
    for (int d = 0; d < n; ++d) bias[3 * H + d] = M->bias[2][d];
    for (int o = 0; o < 4; ++o) bias[3 * H + KO + o] = M->c2[o];

    int dev = 0; cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&P->sms, cudaDevAttrMultiProcessorCount, dev);
    auto up = [](void **dst, const void *src, size_t bytes) {
        return cudaMalloc(dst, bytes ? bytes : 16) == cudaSuccess && (bytes == 0 || cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice) == cudaSuccess);
    };
    bool ok = up(&P->d_wimg, img.data(), img.size()) && up(&P->d_fills, fills.data(), fills.size() * sizeof(uint2)) &&
              up(&P->d_chunks, chunks.data(), chunks.size() * sizeof(ChunkOp)) &&
              up(&P->d_res, res.data(), res.size()) && up(&P->d_bias, bias.data(), bias.size() * 4);
    {   // the attribute belongs to the kernel, not to the model: keep the largest request
        static int max_smem = 0;
        if ((int)P->L.total > max_smem) {
            ok = ok && cudaFuncSetAttribute(eloc_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P->L.total) == cudaSuccess;
            if (ok) max_smem = (int)P->L.total;
        }
    }
    if (!ok) {
        cudaGetLastError();
        cudaFree(P->d_wimg); cudaFree(P->d_fills); cudaFree(P->d_chunks); cudaFree(P->d_res); cudaFree(P->d_bias);
        delete P;
        return NQS_ECUDA;
    }
    M->tc = P;
    return NQS_OK;
}

void tc_pack_free(const nqs_made *M) {
    if (!M->tc) return;
    TcPack *P = M->tc;
    cudaFree(P->d_wimg); cudaFree(P->d_fills); cudaFree(P->d_chunks); cudaFree(P->d_res); cudaFree(P->d_bias);
    if (P->d_fpos) cudaFree(P->d_fpos);
    if (P->d_xpos) cudaFree(P->d_xpos);
    delete P;
    M->tc = nullptr;
}

void tc_mma_counts(const nqs_made *M, long long *issued, long long *dense) {
    *issued = M->tc ? M->tc->mma_issued : 0;
    *dense = M->tc ? M->tc->mma_dense : 0;
}

static void fill_common(const nqs_made *M, TcParams &p) {
    const TcPack *P = M->tc;
    p.n = M->n; p.H = M->h; p.NC = P->NC; p.KI = P->KI; p.KO = P->KO;
    p.tm_d = P->tm_d; p.tm_d3 = P->tm_d3;
    p.wimg = (const uint8_t *)P->d_wimg; p.fills = (const uint2 *)P->d_fills; p.nfills = P->nfills;
    memcpy(p.sub, P->sub, sizeof(p.sub)); memcpy(p.nblk, P->nblk, sizeof(p.nblk));
    p.chunks = (const ChunkOp *)P->d_chunks; p.nchunks = P->nchunks;
    p.resimg = (const uint8_t *)P->d_res; p.res_bytes = P->res_bytes;
    p.slot_bytes = P->slot_bytes; p.nslots = P->nslots;
    p.bias = (const float *)P->d_bias;
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
    // position-ordered flips: rebuilt on the caller's stream for every launch (19 MB of traffic at cfg 5, microseconds
    // next to the chain kernel).  No cache: a device address is not an identity (a freed Hamiltonian's buffers are
    // handed to the next one of the same size), and a cache filled on one stream is unordered against another.
    if ((rc = ensure(&P->d_fpos, &P->fpos_cap, sizeof(ulonglong2) * (size_t)(hm.G ? hm.G : 1)))) return rc;
    if (hm.G > 0 && (rc = permuted(M, hm.flips, hm.G, (ulonglong2 *)P->d_fpos, st))) return rc;
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
