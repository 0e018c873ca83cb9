// Tensor-core path (NQS_PATH_TC): ONE persistent, warp-specialised sm_100a kernel run by CTA PAIRS (clusters of two
// CTAs on one TPC, tcgen05 cta_group::2).  A pair works on two tiles at a time — CTA r on tile 2q + r, a tile being
// 128 samples x 1 unique-flip group g — and every MMA covers both: M = 256 rows (128 per CTA), the weight operand B
// split by rows between the two CTAs' shared memories, so each SM streams only HALF of the weight image.  Per tile:
//   (a2) x' = x xor f_g expanded to a +-1 fp16 operand tile A0, written straight into TENSOR MEMORY (A operand of the
//        input-layer MMAs; no shared-memory copy of the inputs exists),
//   (a4) the MADE chain and the phase MLP as tcgen05 MMAs (fp16 operands, fp32 accumulation in TMEM), in 128-unit
//        hidden CHUNKS that rotate through up to three 128-column TMEM accumulators:
//          layer 1   D = A0 . W1c^T   TS  -> epilogue: ReLU, fp16 -> A1 in SHARED memory (128B-swizzled K-major)
//          phase     D = A0 . P1c^T   TS  -> epilogue: ReLU, fp16 IN PLACE -> D3 += D . P2c^T   (TS, N = 16)
//          layer 2   D = A1 . W2c^T   SS  -> epilogue: ReLU, fp16 IN PLACE -> D3 += D . W3c^T   (TS)
//        (one hidden layer: layer 1 is rewritten in place and feeds W3 directly).  The hidden-layer BIASES are part of
//        the MMAs: A0 carries two constant +1 columns and every weight image two bias columns (fp16 hi + lo parts);
//        layer 2 gets its bias from a one-K-step MMA on A0's constant columns, which also overwrites the accumulator.
//        The chunk epilogue is therefore tcgen05.ld -> cvt.rn.relu.f16x2 -> store, nothing else (the F2FP pipe, 16
//        lanes/clk/SM, is what bounds it).  All-zero K-steps of the masked weights are never issued (exact),
//   (a3) the Pauli contraction S[i,g] over the group's terms (popcount parity, (-i)^r folded into c),
//   (a5) ratio = exp(dlog|psi|) cis(dphi), E_i += S * ratio, kept in registers per sample.
// Warp roles (14 warps per CTA): 12 = weight producer (TMA 1-D bulk copies of this CTA's half of the weight image into
// a ring of two large slots); 13 = in the leader CTA the MMA issuer (ONE elect.sync thread issues every tcgen05.mma /
// commit of the pair; commits are multicast to the barriers of both CTAs), in the peer CTA a forwarder that tells the
// leader when the peer's half of a ring slot has landed; 4-7 / 8-11 = two chunk-epilogue groups, each serving one
// 64-column half of every op; 0-3 = tile warps (A0 of the NEXT tile, contraction, final epilogue).  DESIGN.md 6-7.
// PAPER.md:122-134 (Alg. 1), :84-96 (architecture, Eq. 8-10), :152-158 (Eq. 15-16).
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>
#include "nqs_internal.h"
#include "tc_ptx.cuh"

using namespace tc;

namespace {

constexpr int TILE_M = 128;
constexpr int CN = 128;                  // hidden-unit chunk = accumulator columns = MMA N of the pair
constexpr int HALF = CN / 2;             // weight rows per CTA and chunk
constexpr int NTHREADS = 448;
constexpr int MAX_NC = 4;                // hidden <= 512
constexpr int MAX_SLOTS = 8;
constexpr int NPROD = 4;                 // producer lanes (bulk-copy issuers), never more than slots
constexpr int MAX_OPS = 3 * MAX_NC;
// warp roles.  The warp scheduler of an SM sub-partition (warp id % 4) prefers the HIGHEST warp id among its eligible
// warps, and every sub-partition hosts epilogue warps (a warp reaches only TMEM lane quadrant id % 4): the one thread
// that issues all MMAs therefore lives in the highest warp id of its sub-partition, or it only gets the issue slots
// the epilogue warps leave over.
constexpr int W_EPI = 4, W_PROD = 12, W_ISSUE = 13;      // warps 0-3: tile warps, 4-11: two chunk-epilogue groups (column halves)

enum : uint8_t { T_L1S = 0, T_L1I = 1, T_P = 2, T_L2 = 3 };   // layer 1 -> smem A1 | layer 1 in place | phase hidden | layer 2

// barrier ids.  Waited by the leader's issuer (arrivals from both CTAs): A0FULL, D3EMPTY, EDONE[], WFULL[] (leader copy).
// Committed by the issuer into BOTH CTAs: A0FREE, A1FREE, D3FULL, FULL[], WEMPTY[].
enum { BAR_A0FULL = 0, BAR_A0FREE = 1, BAR_A1FREE = 2, BAR_D3FULL = 3, BAR_D3EMPTY = 4, BAR_FULL = 5, BAR_EDONE = 8,
       BAR_WFULL = 11, BAR_WEMPTY = 11 + MAX_SLOTS, BAR_COUNT = 11 + 2 * MAX_SLOTS };

// Streamed weight sub-tiles: one 32-bit word each, in consumption order (kernel parameter space -> uniform loads).
constexpr int MAX_SUB = 2 * MAX_NC + MAX_NC * (1 + 2 * MAX_NC) + MAX_NC;   // W1 + P1 + (b2 rows + W2 blocks) + W3 (split mode, NC <= 2: fewer)
constexpr uint32_t SUB_OFF_MASK = 0x1FFFu;                   // [0:13)  byte offset inside the slot / 16
constexpr uint32_t SUB_NEW = 1u << 13;                       // first sub-tile of a ring fill: wait for the fill
constexpr uint32_t SUB_END = 1u << 14;                       // last sub-tile of a ring fill: release the slot
constexpr uint32_t SUB_ACC = 1u << 15;                       // input sub-tile: accumulate onto the accumulator (the lo-part pass)
constexpr int SUB_AUX_SHIFT = 16;                            // [16:24) input: K-steps; W2: k-block | K-step mask << 4; W3: n_lo / 16

struct SmemLayout { uint32_t a1, res, bias, bars, slots, total; };

__host__ __device__ inline SmemLayout smem_layout(int H, int KO, int L, uint32_t slot_bytes, int nslots, int split) {
    SmemLayout S;
    uint32_t off = 0;
    const uint32_t parts = split ? 2u : 1u;                          // split precision: hi and lo fp16 parts of everything
    S.a1 = off; if (L == 2) off += parts * (uint32_t)(H / 64) * 16384u;   // fp16 layer-1 activations, K-blocks of 128 rows x 128 B (hi blocks, then lo)
    S.res = off; off += parts * (uint32_t)(H / 64) * 1024u;          // resident P2 tiles: 8 rows x 64 K per K-block (this CTA's half)
    S.bias = off; off += (uint32_t)(KO + 4) * 4;                 // b3 | c2 (hidden-layer biases ride in the weight images)
    off = (off + 15) & ~15u;
    S.bars = off; off += BAR_COUNT * 8;
    off = (off + 1023) & ~1023u;
    S.slots = off; off += slot_bytes * (uint32_t)nslots;
    S.total = off;
    return S;
}

struct TcParams {
    int n, H, NC, KI, KO, L, nacc, nops, split, seq;
    uint32_t tm_d3, tm_a0;               // TMEM columns: accumulator a at a * CN, D3 at tm_d3, A0 at tm_a0
    const uint8_t *wimg; uint32_t img_stride;     // streamed weight image of cluster rank r at wimg + r * img_stride
    const uint2 *fills; int nfills;      // per-tile ring fills (byte offset, bytes), consumption order, same for both ranks
    uint32_t sub[MAX_SUB + 1];
    uint8_t nblk[MAX_NC];                // layer-2 k-blocks issued per output chunk
    uint8_t optype[MAX_OPS], opchunk[MAX_OPS];
    uint8_t prewait[MAX_OPS];            // bit a: wait for the chunk epilogue pending on accumulator a before issuing op j
    uint32_t cntmask;                    // bit a: accumulator a is used an odd number of times per tile
    const uint8_t *resimg; uint32_t res_bytes;    // resident P2 tiles of rank r at resimg + r * res_bytes
    uint32_t slot_bytes; int nslots, nprod;
    const float *bias;                   // [b3 KO | c2 4] fp32
    int mode;                            // 0 = logpsi, 1 = local energy
    const ulonglong2 *xpos;              // [B] configurations, bits in autoregressive POSITION order
    long long B;
    float2 *out;                         // mode 0: (log|psi|, phi) per row
    const ulonglong2 *fpos;              // [G] flips in position order
    const ulonglong2 *x;                 // [B] samples in qubit order (contraction parity)
    HamDev hm;
    const float2 *base;                  // [B] (log|psi|, phi) of the samples
    float2 *epart;                       // [nsb][eslots][TILE_M] per-CTA partial sums of E (slot = 2 * (cluster - first cluster of the block) + rank)
    int eslots;                          // slots per sample block (host: 2 * the largest number of clusters that share a block)
    unsigned *max_ratio_bits;
    long long g_begin;                   // first group that needs a forward pass (1 if group 0 is f = 0)
    int n_up, n_down;                    // Hamming-weight constraint (Eq. 14), n_up < 0 = off
    unsigned long long spin_lo, spin_hi; // bit d = 1: position d is a down spin
};


__device__ __forceinline__ unsigned long long shr128(ulonglong2 a, int s) {      // low 64 bits of a >> s, 0 <= s < 128
    if (s == 0) return a.x;
    if (s < 64) return (a.x >> s) | (a.y << (64 - s));
    return a.y >> (s - 64);
}

// The per-tile op schedule, fixed at compile time so that the issuing thread runs straight-line code (the tensor pipe
// queues only ~100 cycles of MMAs ahead of the issuer, measured).  Two hidden layers: short ops (layer-1 chunk -> A1,
// phase chunk) are interleaved with the long layer-2 chunks, each as early as its inputs allow, so that a chunk
// epilogue (~1 us hand-over round trip) always runs under the MMAs of the next two ops; one hidden layer: layer-1
// chunk c (in place) / phase chunk c alternating.  Op j runs in accumulator j % NACC, whose epilogue group (warps
// W_EPI + 4 a ..) handles every op of that accumulator; the consumer of an in-place op is issued LAG = NACC - 1 ops
// later, just before the accumulator's next producer.
template <int NC, int L, int NACC, bool SEQ>
struct Sched {
    static constexpr int NOPS = (L == 2) ? 3 * NC : 2 * NC;
    static constexpr int LAG = NACC - 1;
    static constexpr int FIRST_INPLACE = (L == 2) ? (SEQ ? NC : (NC > 1 ? 2 : 1)) : 0;
    static constexpr int LAST_A0 = (L == 2) ? NOPS - 2 : NOPS - 1;
    // two hidden layers, interleaved (layer-2 chunk c reads layer-1 chunks <= c only — the sorted-degree masks):
    //     L1S 0 | (L1S c+1, P c, L2 c) for c < NC-1 | P NC-1, L2 NC-1
    // two hidden layers, SEQ (any masks: some layer-2 chunk reads a later layer-1 chunk): every L1S first, then (P c, L2 c)
    __host__ __device__ static constexpr int type(int j) {
        if (L != 2) return (j & 1) ? (int)T_P : (int)T_L1I;
        if (SEQ) return j < NC ? (int)T_L1S : (((j - NC) & 1) ? (int)T_L2 : (int)T_P);
        if (j == 0) return (int)T_L1S;
        const int jj = j - 1;
        if (jj < 3 * (NC - 1)) return jj % 3 == 0 ? (int)T_L1S : (jj % 3 == 1 ? (int)T_P : (int)T_L2);
        return (jj - 3 * (NC - 1)) == 0 ? (int)T_P : (int)T_L2;
    }
    __host__ __device__ static constexpr int chunk(int j) {
        if (L != 2) return j / 2;
        if (SEQ) return j < NC ? j : (j - NC) / 2;
        if (j == 0) return 0;
        const int jj = j - 1;
        if (jj < 3 * (NC - 1)) return jj % 3 == 0 ? jj / 3 + 1 : jj / 3;
        return NC - 1;
    }
};

template <int NC, int L, int NACC, bool SPLIT, bool SEQ>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NTHREADS, 1) eloc_tc_kernel(const __grid_constant__ TcParams p) {
    using S = Sched<NC, L, NACC, SEQ>;
    extern __shared__ __align__(1024) uint8_t smem[];
    __shared__ uint32_t s_tmem_base;
    const SmemLayout SL = smem_layout(p.H, p.KO, p.L, p.slot_bytes, p.nslots, SPLIT ? 1 : 0);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + SL.bars);
    float *s_bias = reinterpret_cast<float *>(smem + SL.bias);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const int KI = p.KI, KO = p.KO;
    constexpr uint32_t nops = S::NOPS;
    const uint32_t smem_base = smem_u32(smem);
    const uint32_t bars_addr = smem_base + SL.bars;
#define BAR_ADDR(id) (bars_addr + (uint32_t)(id) * 8u)

    // ---- one-time setup ----
    if (threadIdx.x == 0) {
        mbar_init(&bars[BAR_A0FULL], 8); mbar_init(&bars[BAR_A0FREE], 1); mbar_init(&bars[BAR_A1FREE], 1);
        mbar_init(&bars[BAR_D3FULL], 1); mbar_init(&bars[BAR_D3EMPTY], 8);
        for (int a = 0; a < 3; ++a) { mbar_init(&bars[BAR_FULL + a], 1); mbar_init(&bars[BAR_EDONE + a], 16); }   // 8 epilogue warps x 2 CTAs
        for (int s = 0; s < p.nslots; ++s) {
            mbar_init(&bars[BAR_WFULL + s], rank == 0 ? 2 : 1);      // leader: own producer + the peer's forwarder
            mbar_init(&bars[BAR_WEMPTY + s], 1);
        }
        fence_mbar_init();
    }
    if (warp == W_ISSUE) tmem_alloc_cg2(&s_tmem_base, 512);
    for (int i = threadIdx.x; i < KO + 4; i += NTHREADS) s_bias[i] = p.bias[i];
    for (int i = threadIdx.x; i < (int)(p.res_bytes / 16); i += NTHREADS)
        reinterpret_cast<uint4 *>(smem + SL.res)[i] = reinterpret_cast<const uint4 *>(p.resimg + (size_t)rank * p.res_bytes)[i];
    fence_proxy_async();                                  // resident tiles are read by the tensor core (async proxy)
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem = s_tmem_base;

    // ---- static schedule: a contiguous range of tile PAIRS per cluster, sample-block major; CTA r takes tile 2q + r ----
    const long long nsb = (p.B + TILE_M - 1) / TILE_M;
    const long long Gnd = (p.mode == 1) ? (p.hm.G - p.g_begin) : 1;
    const long long ntiles = nsb * Gnd;
    const long long npairs = (ntiles + 1) / 2;
    const long long ncl = gridDim.x >> 1, cl = blockIdx.x >> 1;
    const long long q_lo = npairs * cl / ncl, q_hi = npairs * (cl + 1) / ncl;
    const long long ntl = q_hi - q_lo;

    if (warp == W_PROD) {
        // =========================== weight producers (TMA engine, 1-D bulk copies), both CTAs ===========================
        // Fill q always lands in slot q % nslots.  Never more lanes than slots: a lane two uses of a slot ahead of the
        // consumer would pass its parity wait on an older phase and overwrite live data.
        const uint32_t nprod = (uint32_t)p.nprod;
        if ((uint32_t)lane < nprod) {
            const long long total = ntl * (long long)p.nfills;
            const uint8_t *img = p.wimg + (size_t)rank * p.img_stride;
            uint32_t e = (uint32_t)lane % (uint32_t)p.nfills, slot = (uint32_t)lane, par = 1u;   // a fresh barrier passes a parity-1 wait
            for (long long q = lane; q < total; q += nprod) {
                const uint2 pe = __ldg(&p.fills[e]);
                mbar_wait(&bars[BAR_WEMPTY + slot], par);
                mbar_arrive_expect_tx(&bars[BAR_WFULL + slot], pe.y);
                bulk_g2s(smem + SL.slots + slot * p.slot_bytes, img + pe.x, pe.y, &bars[BAR_WFULL + slot]);
                e += nprod; while (e >= (uint32_t)p.nfills) e -= (uint32_t)p.nfills;
                slot += nprod; while (slot >= (uint32_t)p.nslots) { slot -= (uint32_t)p.nslots; par ^= 1u; }
            }
        }
    } else if (warp == W_ISSUE && rank != 0) {
        // =========================== peer CTA: ring forwarder ===========================
        // The leader's MMAs read this CTA's half of every ring slot; a bulk copy can only signal a barrier of its own
        // CTA, so one thread waits for each local fill and arrives on the leader's WFULL barrier of the same slot.
        if (elect_one()) {
            const long long total = ntl * (long long)p.nfills;
            uint32_t slot = 0, par = 0;
            for (long long q = 0; q < total; ++q) {
                mbar_wait(&bars[BAR_WFULL + slot], par);
                mbar_arrive_cluster(BAR_ADDR(BAR_WFULL + slot), 0);
                if (++slot == (uint32_t)p.nslots) { slot = 0; par ^= 1u; }
            }
        }
        __syncwarp();
    } else if (warp == W_ISSUE) {
        // =========================== leader CTA: MMA issuer, ONE elected thread ===========================
        // Ops of a tile are issued in the fixed order of Sched; the consumer of an in-place op (P2 / W3 MMAs reading the
        // fp16 chunk the epilogue wrote over the accumulator) is issued LAG ops later — the tensor pipe executes in
        // issue order, so MMA-after-MMA hazards need no barrier; only epilogue <-> MMA hand-overs do (FULL / EDONE).
        // Every EDONE phase is waited exactly once, at a position fixed on the host (p.prewait) or at the consumer, so
        // barrier parities are plain bits of `ph`.
        if (elect_one()) {
            const uint32_t a1_lo = (smem_base + SL.a1) >> 4, res_lo = (smem_base + SL.res) >> 4;
            const uint32_t slots_lo = (smem_base + SL.slots) >> 4, slot_step = p.slot_bytes >> 4;
            // descriptor words: lo = addr/16 | (lbo/16) << 16, hi = sbo/16 | version 1 << 14 | layout << 29
            const uint32_t lo_noswz = (128u >> 4) << 16, hi_noswz = (((uint32_t)(KI / 8) * 128u) >> 4) | (1u << 14);
            const uint32_t hi_noswz16 = (256u >> 4) | (1u << 14);          // one K-step wide tile (the layer-2 bias rows)
            const uint32_t lo_sw128 = (16u >> 4) << 16, hi_sw128 = (1024u >> 4) | (1u << 14) | (2u << 29);
            const uint32_t id128 = idesc_f16(256, CN), id16 = idesc_f16(256, 16), id0 = idesc_f16(256, 0);
            const uint32_t nslots = (uint32_t)p.nslots;
            const uint32_t tm_d3 = tmem + p.tm_d3, tm_ph = tm_d3 + (uint32_t)KO - 16, tm_a0 = tmem + p.tm_a0;
            uint32_t slot = 0, wpar = 0, slot_lo = slots_lo;
            uint32_t ph = 0;                             // parity of the next phase to wait for, one bit per barrier id
#define WAIT(id) do { mbar_spin(BAR_ADDR(id), (ph >> (id)) & 1u); ph ^= 1u << (id); tc_fence_after(); } while (0)
#define SLOT_ACQUIRE(w) do { if ((w) & SUB_NEW) { mbar_spin(BAR_ADDR(BAR_WFULL + slot), wpar); tc_fence_after(); } } while (0)
#define SLOT_RELEASE(w) do { if ((w) & SUB_END) { mma_commit_cg2(BAR_ADDR(BAR_WEMPTY + slot)); slot_lo += slot_step; \
                             if (++slot == nslots) { slot = 0; wpar ^= 1u; slot_lo = slots_lo; } } } while (0)
            for (long long ti = 0; ti < ntl; ++ti) {
                // (the table index goes through an opaque asm so that the compiler cannot prove the table words loop-invariant
                // and unswitch the tile loop on them: that multiplied the issuer's code size by ten)
                uint32_t si = 0;
                asm volatile("" : "+r"(si));
                uint32_t w = p.sub[si];                      // current table word; the next one is always loaded one step ahead
                WAIT(BAR_A0FULL);
                // consumer of tile-local op jc (jc is a compile-time constant after unrolling)
                auto consume = [&](const int jc) {
                    const int type = S::type(jc);
                    if (type == T_L1S) return;
                    // every address is computed and the weight slot acquired BEFORE the wait for the chunk epilogue, so
                    // that the first MMA leaves right behind the poll (an idle pipe costs ~100 cycles to restart)
                    const uint32_t a_t = tmem + (uint32_t)(jc % NACC) * CN;
                    // split precision: the epilogue left fp16 hi parts in columns [32 pc, 32 pc + 16) and lo parts in
                    // [32 pc + 16, 32 pc + 32) of every 32-column piece; D3 += Ahi.Bhi + Alo.Bhi + Ahi.Blo
                    if (type == T_P) {                                          // resident P2 tile of this chunk, N = 16
                        const uint32_t b_lo = (res_lo + (uint32_t)S::chunk(jc) * ((SPLIT ? 4096u : 2048u) >> 4)) | lo_sw128;
                        WAIT(BAR_EDONE + jc % NACC);
                        if (jc == S::FIRST_INPLACE) { WAIT(BAR_D3EMPTY); }          // first write into D3 of this tile
#pragma unroll
                        for (uint32_t ks = 0; ks < 8; ++ks) {
                            const uint32_t a_k = a_t + 32 * (ks >> 1) + 8 * (ks & 1), b_k = b_lo + (ks >> 2) * (1024u >> 4) + 2 * (ks & 3);
                            mma_ts_cg2(tm_ph, a_k, b_k, hi_sw128, id16, 1u);
                            if (SPLIT) {
                                mma_ts_cg2(tm_ph, a_k + 16, b_k, hi_sw128, id16, 1u);
                                mma_ts_cg2(tm_ph, a_k, b_k + (2048u >> 4), hi_sw128, id16, 1u);
                            }
                        }
                    } else {                                                    // streamed layer-3 tile
                        const uint32_t wn = p.sub[++si];
                        const uint32_t nlo = ((w >> SUB_AUX_SHIFT) & 0xFFu) * 16;      // output rows below n_lo receive exactly 0
                        const uint32_t N = (uint32_t)KO - nlo, kb_step = (N >> 1) * (128u >> 4);
                        const uint32_t b_lo = (slot_lo + (w & SUB_OFF_MASK)) | lo_sw128, idesc = id0 | ((N >> 3) << 17);
                        SLOT_ACQUIRE(w);
                        WAIT(BAR_EDONE + jc % NACC);
                        if (jc == S::FIRST_INPLACE) { WAIT(BAR_D3EMPTY); }          // first write into D3 of this tile
#pragma unroll
                        for (uint32_t ks = 0; ks < 8; ++ks) {
                            const uint32_t a_k = a_t + 32 * (ks >> 1) + 8 * (ks & 1), b_k = b_lo + (ks >> 2) * kb_step + 2 * (ks & 3);
                            mma_ts_cg2(tm_d3 + nlo, a_k, b_k, hi_sw128, idesc, 1u);
                            if (SPLIT) {
                                mma_ts_cg2(tm_d3 + nlo, a_k + 16, b_k, hi_sw128, idesc, 1u);
                                mma_ts_cg2(tm_d3 + nlo, a_k, b_k + 2 * kb_step, hi_sw128, idesc, 1u);      // lo-part tile: N * 128 bytes on
                            }
                        }
                        SLOT_RELEASE(w);
                        w = wn;
                    }
                };
#pragma unroll
                for (int j = 0; j < S::NOPS; ++j) {
                    const int type = S::type(j), c = S::chunk(j), acc = j % NACC;
                    uint32_t jj = (uint32_t)j;
                    asm volatile("" : "+r"(jj));
                    const uint32_t pw = p.prewait[jj];      // pending chunk epilogues this op depends on (accumulator reuse, A1 chunks)
                    if (pw & 1u) WAIT(BAR_EDONE + 0);
                    if (NACC > 1 && (pw & 2u)) WAIT(BAR_EDONE + 1);
                    if (NACC > 2 && (pw & 4u)) WAIT(BAR_EDONE + 2);
                    const uint32_t d = tmem + (uint32_t)acc * CN;
                    if (type == T_L2) {
                        const uint32_t nb = p.nblk[jj - (uint32_t)(j - c)];
                        {   // D = [1 1 x'..] . [b2_hi b2_lo 0..]^T: the bias, and the overwrite of the accumulator
                            const uint32_t wn = p.sub[++si];
                            SLOT_ACQUIRE(w);
                            mma_ts_cg2(d, tm_a0, (slot_lo + (w & SUB_OFF_MASK)) | lo_noswz, hi_noswz16, id128, 0u);
                            SLOT_RELEASE(w);
                            w = wn;
                        }
                        if (j == S::NOPS - 1) mma_commit_cg2(BAR_ADDR(BAR_A0FREE));            // last reader of A0 in a two-layer tile
                        const uint32_t accum = 1u;
#pragma unroll 1
                        for (uint32_t b = 0; b < nb; ++b) {
                            const uint32_t wn = p.sub[++si];
                            SLOT_ACQUIRE(w);
                            const uint32_t aux = (w >> SUB_AUX_SHIFT) & 0xFFu, kmask = aux >> 4;
                            const uint32_t a_lo = (a1_lo + (aux & 7u) * (16384u >> 4)) | lo_sw128;
                            const uint32_t b_lo = (slot_lo + (w & SUB_OFF_MASK)) | lo_sw128;
                            if (kmask == 0xFu) {
                                mma_ss_cg2(d, a_lo, hi_sw128, b_lo, hi_sw128, id128, accum);
                                mma_ss_cg2(d, a_lo + 2, hi_sw128, b_lo + 2, hi_sw128, id128, 1u);
                                mma_ss_cg2(d, a_lo + 4, hi_sw128, b_lo + 4, hi_sw128, id128, 1u);
                                mma_ss_cg2(d, a_lo + 6, hi_sw128, b_lo + 6, hi_sw128, id128, 1u);
                            } else {
#pragma unroll
                                for (uint32_t ks = 0; ks < 4; ++ks)
                                    if ((kmask >> ks) & 1u) mma_ss_cg2(d, a_lo + 2 * ks, hi_sw128, b_lo + 2 * ks, hi_sw128, id128, accum);
                            }
                            if (SPLIT && (w & SUB_ACC)) {       // the hi weight block serves the lo activations too (H/64 k-blocks on)
                                const uint32_t a_l2 = a_lo + (uint32_t)(p.H / 64) * (16384u >> 4);
#pragma unroll
                                for (uint32_t ks = 0; ks < 4; ++ks)
                                    if ((kmask >> ks) & 1u) mma_ss_cg2(d, a_l2 + 2 * ks, hi_sw128, b_lo + 2 * ks, hi_sw128, id128, accum);
                            }
                            SLOT_RELEASE(w);
                            w = wn;
                        }
                    } else {
                        // input layers (layer 1 / phase hidden): A = A0 in TMEM (exact +-1), B = this chunk's rows, K-step
                        // prefix; split precision: a second pass over the same A with the lo parts of the weights
#pragma unroll
                        for (int part = 0; part < (SPLIT ? 2 : 1); ++part) {
                            const uint32_t wn = p.sub[++si];
                            SLOT_ACQUIRE(w);
                            const uint32_t nk = (w >> SUB_AUX_SHIFT) & 0xFFu;
                            const uint32_t b_lo = (slot_lo + (w & SUB_OFF_MASK)) | lo_noswz;
                            mma_ts_cg2(d, tm_a0, b_lo, hi_noswz, id128, (uint32_t)part);
                            // nested so that the common exit is one taken branch (KI <= 128 -> at most 8 K-steps)
#define KSTEP(k) mma_ts_cg2(d, tm_a0 + 8u * (k), b_lo + 16u * (k), hi_noswz, id128, 1u)
                            if (nk > 1) { KSTEP(1); if (nk > 2) { KSTEP(2); if (nk > 3) { KSTEP(3); if (nk > 4) { KSTEP(4);
                            if (nk > 5) { KSTEP(5); if (nk > 6) { KSTEP(6); if (nk > 7) { KSTEP(7); } } } } } } }
#undef KSTEP
                            SLOT_RELEASE(w);
                            w = wn;
                        }
                    }
                    mma_commit_cg2(BAR_ADDR(BAR_FULL + acc));
                    if (L == 1 && j == S::LAST_A0) mma_commit_cg2(BAR_ADDR(BAR_A0FREE));       // A0 may be rebuilt for the next tile
                    if (L == 2 && j == S::NOPS - 1) mma_commit_cg2(BAR_ADDR(BAR_A1FREE));      // A1 may be rewritten by the next tile
                    if (j >= S::LAG) consume(j - S::LAG);
                }
#pragma unroll
                for (int m = S::LAG; m >= 1; --m) consume(S::NOPS - m);                       // consumers of the last ops
                mma_commit_cg2(BAR_ADDR(BAR_D3FULL));
            }
#undef WAIT
#undef SLOT_ACQUIRE
#undef SLOT_RELEASE
        }
        __syncwarp();
    } else if (warp >= W_EPI) {
        // =========================== chunk epilogue groups: ops alternate between the two groups ===========================
        // Every op is served by BOTH groups, each taking one half of the accumulator's columns (two 32-column pieces), so
        // that the hand-over round trip commit -> epilogue -> arrive is half as long.  An in-place op keeps each piece's
        // fp16 result inside the piece's own columns [32 pc, 32 pc + 16): no piece ever writes what another still reads.
        const uint32_t grp = (uint32_t)(warp - W_EPI) >> 2;
        const uint32_t row = (uint32_t)((warp & 3) * 32 + lane);
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;     // TMEM lane quadrant of this warp
        const uint32_t a1_row = smem_base + SL.a1 + (row >> 3) * 1024u + (row & 7u) * 128u, sw = row & 7u;
        uint32_t fb = 0;                                   // bit a: parity of accumulator a's first FULL phase of this tile
        for (long long ti = 0; ti < ntl; ++ti, fb ^= p.cntmask) {
        bool a1_waited = false;
        uint32_t acc = 0, q = 0;                           // j % NACC, j / NACC
        for (uint32_t j = 0; j < nops; ++j) {
            const uint32_t type = p.optype[j], c = p.opchunk[j];
            mbar_wait(&bars[BAR_FULL + acc], ((fb >> acc) ^ q) & 1u);
            tc_fence_after();
            // before the first write into A1: the previous tile's layer-2 MMAs have read it
            if (L == 2 && ti > 0 && type == T_L1S && !a1_waited) {
                mbar_wait(&bars[BAR_A1FREE], (uint32_t)(ti - 1) & 1u);
                a1_waited = true;
            }
            const uint32_t d_addr = tmem + lane_base + acc * CN + 64u * grp;
            uint32_t va[32], vb[32];
            tmem_ld32p(d_addr, va);
            tmem_ld32p(d_addr + 32, vb);
            tmem_wait_ld();
#pragma unroll
            for (int pp = 0; pp < 2; ++pp) {
                const uint32_t *v = pp ? vb : va;
                uint32_t w[16], wl[16];                        // the bias is already in the accumulator (constant input columns)
#pragma unroll
                for (int j2 = 0; j2 < 16; ++j2) {
                    const float x0 = __uint_as_float(v[2 * j2]), x1 = __uint_as_float(v[2 * j2 + 1]);
                    w[j2] = cvt_relu_f16x2(x0, x1);
                    if (SPLIT) {                               // lo part: what the fp16 rounding of relu(x) lost, again as fp16
                        const float2 hf = __half22float2(*reinterpret_cast<const __half2 *>(&w[j2]));
                        wl[j2] = cvt_f16x2(fmaxf(x0, 0.0f) - hf.x, fmaxf(x1, 0.0f) - hf.y);
                    }
                }
                if (type == T_L1S) {
                    // this group's 64 hidden units are K-block 2c + grp of A1; 32 units = four 16-byte pieces, 128B swizzle
                    const uint32_t kb_addr = a1_row + (2 * c + grp) * 16384u;
#pragma unroll
                    for (uint32_t i = 0; i < 4; ++i) {
                        const uint32_t jj = (uint32_t)pp * 4 + i;
                        st_shared_v4(kb_addr + ((jj ^ sw) << 4), w[4 * i], w[4 * i + 1], w[4 * i + 2], w[4 * i + 3]);
                        if (SPLIT) st_shared_v4(kb_addr + (uint32_t)(p.H / 64) * 16384u + ((jj ^ sw) << 4), wl[4 * i], wl[4 * i + 1], wl[4 * i + 2], wl[4 * i + 3]);
                    }
                } else {
                    tmem_st16p(d_addr + 32 * pp, w);          // in place, inside the piece's own columns
                    if (SPLIT) tmem_st16p(d_addr + 32 * pp + 16, wl);
                }
            }
            if (type == T_L1S) fence_proxy_async(); else tmem_wait_st();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_leader(BAR_ADDR(BAR_EDONE + acc), rank);
            __syncwarp();
            if (++acc == (uint32_t)NACC) { acc = 0; ++q; }
        }
        }
    } else {
        // =========================== tile warps: A0 of the next tile, contraction, final epilogue ===========================
        const int q = warp & 3;
        const int row = q * 32 + lane;
        const uint32_t lane_base = (uint32_t)(q * 32) << 16;
        const uint32_t d3_addr = tmem + lane_base + p.tm_d3, a0_addr = tmem + lane_base + p.tm_a0;
        const float *s_b3 = s_bias, *s_c2 = s_bias + KO;
        const uint32_t zero16[16] = {0};

        struct RowState { long long sb, i; ulonglong2 xp, xq; float2 b0; };
        auto load_row = [&](long long sb, bool valid, RowState &r) {
            r.sb = sb; r.i = valid ? sb * TILE_M + row : p.B;
            if (r.i < p.B) {
                r.xp = p.xpos[r.i];
                if (p.mode == 1) { r.xq = p.x[r.i]; r.b0 = p.base[r.i]; }
                else { r.xq = make_ulonglong2(0, 0); r.b0 = make_float2(0.f, 0.f); }
            } else { r.i = p.B; r.xp = make_ulonglong2(0, 0); r.xq = r.xp; r.b0 = make_float2(0.f, 0.f); }
        };
        // (a2) A0: +-1 fp16, one row per thread = one TMEM lane, 16 inputs = 8 columns per K-step
        // K index 0 and 1 are the constant +1 columns that carry the hidden-layer biases (hi + lo fp16 parts); position d
        // of the configuration sits at K index d + 2
        auto build_a0 = [&](ulonglong2 zq) {
            const ulonglong2 zp = make_ulonglong2((zq.x << 2) | 3ull, (zq.y << 2) | (zq.x >> 62));
            for (int kc = 0; kc < KI / 16; ++kc) {
                const uint32_t bits = (uint32_t)(shr128(zp, kc * 16) & 0xFFFFull);
                uint32_t w[8];
#pragma unroll
                for (int jj = 0; jj < 8; ++jj)
                    w[jj] = 0xBC00BC00u ^ (((bits >> (2 * jj)) & 1u) << 15) ^ (((bits >> (2 * jj + 1)) & 1u) << 31);
                tmem_st8p(a0_addr + 8 * kc, w);
            }
            tmem_wait_st();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_leader(BAR_ADDR(BAR_A0FULL), rank);
        };
        auto flip_of = [&](long long t, bool valid) -> ulonglong2 {
            if (p.mode != 1 || !valid) return make_ulonglong2(0, 0);
            return __ldg(&p.fpos[p.g_begin + (t % Gnd)]);
        };

        // D3 accumulates from zero (every MMA into it has accumulate = 1)
        for (int c = 0; c < KO; c += 16) tmem_st16p(d3_addr + c, zero16);
        tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_leader(BAR_ADDR(BAR_D3EMPTY), rank);

        RowState cur{}, nxt{};
        ulonglong2 zp = make_ulonglong2(0, 0), zp_n = zp;
        // Eq. 14: positions whose conditional is clamped contribute log 1 = 0; a string that violates Eq. 12 has psi = 0
        ulonglong2 fm = make_ulonglong2(0, 0), fm_n = fm;
        bool inval = false, inval_n = false;
        auto clamp_of = [&](ulonglong2 z, ulonglong2 &f, bool &bad) {
            if (p.n_up < 0) return;
            bool ok;
            f = nqs_forced_mask(z, p.n, p.spin_lo, p.spin_hi, p.n_up, p.n_down, &ok);
            bad = !ok;
        };
        float2 E = make_float2(0.f, 0.f);
        float mr = (p.mode == 1 && p.hm.has_diag) ? 1.0f : 0.0f;     // the f = 0 group has ratio exactly 1
        if (ntl > 0) {
            const long long t = 2 * q_lo + rank;
            const bool valid = t < ntiles;
            load_row(t / Gnd, valid, cur);
            const ulonglong2 f = flip_of(t, valid);
            zp = make_ulonglong2(cur.xp.x ^ f.x, cur.xp.y ^ f.y);
            clamp_of(zp, fm, inval);
            build_a0(zp);
        }
        for (long long ti = 0; ti < ntl; ++ti) {
            const long long t = 2 * (q_lo + ti) + rank;
            const bool valid = t < ntiles;
            const long long g = p.g_begin + (t % Gnd);
            const bool has_next = ti + 1 < ntl;
            if (has_next) {
                const long long tn = t + 2;
                const bool validn = tn < ntiles;
                const long long sbn = tn / Gnd;
                if (sbn != cur.sb || !validn) load_row(sbn, validn, nxt); else nxt = cur;
                const ulonglong2 f = flip_of(tn, validn);
                zp_n = make_ulonglong2(nxt.xp.x ^ f.x, nxt.xp.y ^ f.y);
                clamp_of(zp_n, fm_n, inval_n);
            }
            // ---- (a3) S = sum_{t in g} c_t (-i)^{r_t} (-1)^{popcount(x & s_t)}: independent of the MMAs, done while they run ----
            float2 S = make_float2(0.f, 0.f);
            if (p.mode == 1 && valid && cur.i < p.B) {
                const uint32_t t1 = __ldg(&p.hm.offsets[g + 1]);
                for (uint32_t tt = __ldg(&p.hm.offsets[g]); tt < t1; ++tt) {
                    const ulonglong2 zy = __ldg(&p.hm.zy[tt]);
                    const float2 c = __ldg(&p.hm.cph[tt]);
                    const float2 cs = nqs_signed(c, nqs_parity_sign(cur.xq, zy));
                    S.x += cs.x;
                    S.y += cs.y;
                }
            }
            // ---- operand tile of the NEXT tile, once the last MMA that reads the current one has completed ----
            if (has_next) {
                mbar_wait(&bars[BAR_A0FREE], (uint32_t)ti & 1u);
                tc_fence_after();
                build_a0(zp_n);
            }
            // ---- final epilogue: log|psi| = 1/2 sum_d log sigmoid(+-a_d), phi = o[2 z_{n-2} + z_{n-1}] ----
            mbar_wait(&bars[BAR_D3FULL], (uint32_t)ti & 1u);
            tc_fence_after();
            // sum_d log sigmoid(t_d) = sum_d min(t_d, 0) - ln prod_d (1 + exp(-|t_d|)): every factor is in (1, 2], so a
            // 16-term product cannot overflow and costs one LG2 per 16 conditionals; the 16 chains are independent (ILP).
            float msum = 0.0f, lg = 0.0f, phi = 0.0f;
            for (int c0 = 0; c0 < KO; c0 += 16) {
                uint32_t v[16];
                tmem_ld16p(d3_addr + c0, v);
                tmem_wait_ld();
                tmem_st16p(d3_addr + c0, zero16);              // D3 restarts from zero for the next tile
                if (c0 + 16 >= KO) {
                    const int sel = (int)((shr128(zp, p.n - 2) & 1ull) * 2 + (shr128(zp, p.n - 1) & 1ull));
                    const float o0 = __uint_as_float(v[12]) + s_c2[0], o1 = __uint_as_float(v[13]) + s_c2[1];
                    const float o2 = __uint_as_float(v[14]) + s_c2[2], o3 = __uint_as_float(v[15]) + s_c2[3];
                    phi = sel == 0 ? o0 : (sel == 1 ? o1 : (sel == 2 ? o2 : o3));
                }
                const uint32_t zb = (uint32_t)shr128(zp, c0), fb = (uint32_t)shr128(fm, c0);
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
                        float tt = ((zb >> k) & 1u) ? a : -a;
                        tt = (k < nv && !((fb >> k) & 1u)) ? tt : 1e30f;      // padding column or clamped conditional: factor 1, min 0
                        const float e = ex2_ftz(fabsf(tt) * -1.4426950408889634f);
                        if (k & 1) { prod1 *= 1.0f + e; m1 += fminf(tt, 0.0f); }
                        else       { prod0 *= 1.0f + e; m0 += fminf(tt, 0.0f); }
                    }
                }
                msum += m0 + m1;
                lg += lg2_ftz(prod0 * prod1);
            }
            const float part = msum - 0.6931471805599453f * lg;
            tmem_wait_st();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_leader(BAR_ADDR(BAR_D3EMPTY), rank);
            const float lp = inval ? -INFINITY : 0.5f * part;
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
            if (!has_next || nxt.sb != cur.sb || nxt.i != cur.i) {
                if (p.mode == 1 && cur.i < p.B) {
                    // One slot per (sample block, CTA): every row's partial is WRITTEN once and eloc_finish_kernel adds
                    // the slots in order, so E_loc does not depend on how the CTAs were scheduled (no float atomics).
                    // The clusters that share block sb are consecutive; the first is the one holding tile pair sb*Gnd/2.
                    const long long k_first = ((((cur.sb * Gnd) >> 1) + 1) * ncl - 1) / npairs;
                    p.epart[((size_t)cur.sb * p.eslots + 2 * (size_t)(cl - k_first) + rank) * TILE_M + row] = E;
                }
                E = make_float2(0.f, 0.f);
            }
            cur = nxt; zp = zp_n; fm = fm_n; inval = inval_n;
        }
        if (p.mode == 1) atomicMax(p.max_ratio_bits, __float_as_uint(mr));
    }
#undef BAR_ADDR
    tc_fence_before();
    cluster_sync_all();
    if (warp == W_ISSUE) tmem_dealloc_cg2(tmem, 512);
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

// eloc[i] = S[i, group 0] (when group 0 is the f = 0 group: psi ratio == 1) + the per-CTA partial sums of the chain
// kernel, added in slot order = cluster order, rank 0 before rank 1: a fixed order, so the result is bit-reproducible.
// Slots no CTA owns were zeroed before the chain kernel ran.
__global__ void eloc_finish_kernel(HamDev hm, const ulonglong2 *__restrict__ x, long long B, const float2 *__restrict__ epart,
                                   int eslots, float2 *__restrict__ eloc) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= B) return;
    float2 S = make_float2(0.f, 0.f);
    if (hm.has_diag) {
        const ulonglong2 xr = x[i];
        const uint32_t t1 = hm.offsets[1];
        for (uint32_t t = hm.offsets[0]; t < t1; ++t) {
            const ulonglong2 zy = __ldg(&hm.zy[t]);
            const float2 c = __ldg(&hm.cph[t]);
            const float2 cs = nqs_signed(c, nqs_parity_sign(xr, zy));
            S.x += cs.x;
            S.y += cs.y;
        }
    }
    const float2 *pp = epart + (size_t)(i / TILE_M) * eslots * TILE_M + (i % TILE_M);
    for (int j = 0; j < eslots; ++j) {
        const float2 e = pp[(size_t)j * TILE_M];
        S.x += e.x;
        S.y += e.y;
    }
    eloc[i] = S;
}

}  // namespace

// ------------------------------------------------------------------------------------------------------------
struct TcPack {
    int KI = 0, KO = 0, NC = 0, nacc = 0, nops = 0, nsub = 0, nfills = 0, nslots = 0, split = 0, Hp = 0, seq = 0;
    uint32_t slot_bytes = 0, res_bytes = 0, img_stride = 0, tm_d3 = 0, tm_a0 = 0;
    void *d_wimg = nullptr, *d_fills = nullptr, *d_res = nullptr, *d_bias = nullptr;
    void *d_fpos = nullptr; size_t fpos_cap = 0;
    void *d_epart = nullptr; size_t epart_cap = 0;   // per-CTA partial sums of E (launch_eloc_tc)
    void *d_xpos = nullptr; size_t xpos_cap = 0;
    SmemLayout L{};
    uint32_t sub[MAX_SUB + 1] = {0};
    uint8_t nblk[MAX_NC] = {0}, l2need[MAX_NC] = {0}, optype[MAX_OPS] = {0}, opchunk[MAX_OPS] = {0}, prewait[MAX_OPS] = {0};
    uint32_t cntmask = 0;
    int sms = 148;
    long long mma_issued = 0, mma_dense = 0;                   // 16-wide K-steps x N issued / of the dense chain, per tile (MACs / 2048)
};

static inline int round16(int v) { return (v + 15) / 16 * 16; }

struct TcShape { int KI, KO, NC, nacc, nslots, split, Hp; uint32_t slot; };

static bool tc_shape(const nqs_made *M, TcShape *out) {
    if ((M->L != 1 && M->L != 2) || M->h < 1 || M->h > CN * MAX_NC) return false;
    TcShape s;
    // the hidden width is padded to a multiple of 128 with units whose weights and biases are zero: relu(0) = 0 feeds
    // zero weights, so the padded network computes exactly the same function
    s.Hp = (M->h + CN - 1) / CN * CN;
    s.KI = round16(M->n + 2); s.KO = round16(M->n + 4); s.NC = s.Hp / CN;      // + 2: the constant bias columns
    // Split precision (every fp16 operand as hi + lo, three MMA passes: hi.hi + lo.hi + hi.lo) where single-pass fp16 misses
    // the 1e-5 sum|c| bound (hidden < 384); the hi/lo activations need twice the A1 width, <= 512
    s.split = (s.Hp <= 256) ? 1 : 0;
    if (s.KI > 128 || s.KO > 144) return false;
    // TMEM: nacc accumulators of CN columns, D3 (KO), A0 (KI/2)
    s.nacc = 3;
    if (s.nacc * CN + s.KO + s.KI / 2 > 512) s.nacc = 2;
    if (s.nacc * CN + s.KO + s.KI / 2 > 512) return false;
    uint32_t need = (uint32_t)HALF * s.KI * 2;                                 // input sub-tile (64 rows x KI)
    if ((uint32_t)HALF * 128 > need) need = HALF * 128;                        // layer-2 sub-tile (64 x 64)
    if ((uint32_t)s.KO * 128 * (1 + s.split) > need) need = (uint32_t)s.KO * 128 * (1 + s.split);   // layer-3 tile (KO/2 rows x 128 K; hi + lo)
    const uint32_t budget = 227 * 1024 - 1024;
    const uint32_t fixed = smem_layout(s.Hp, s.KO, M->L, 0, 0, s.split).total;
    if (fixed + 2 * need > budget) return false;
    const uint32_t ring = budget - fixed;
    // Two large slots (plain double buffering).  Measured: a bulk copy costs its issuing warp ~590 cycles whatever its size
    // (2 KB .. 64 KB), and every hand-over costs the MMA issuer ~220 cycles, so fewer and larger fills win: 2 x 40 KB ran
    // 4 % faster than 4 x 20 KB and 16 % faster than 8 x 10 KB on the 76-qubit workload.
    int ns = 2;
    uint32_t slot = (ring / ns) / 1024 * 1024;
    if (slot < need) return false;
    if (slot > 0x1FFFu * 16u) slot = 0x1FFFu * 16u / 1024 * 1024;
    s.slot = slot; s.nslots = ns;
    *out = s;
    return true;
}

bool tc_supported(const nqs_made *M) {
    TcShape s;
    return tc_shape(M, &s);
}

static inline uint32_t noswz_offset(uint32_t r, uint32_t k, uint32_t KI) {
    return (r >> 3) * (KI / 8) * 128u + (k >> 3) * 128u + (r & 7u) * 16u + (k & 7u) * 2u;
}

int tc_pack_upload(const nqs_made *M) {
    if (M->tc) return NQS_OK;
    TcShape sh;
    if (!tc_shape(M, &sh)) return NQS_EUNSUPPORTED;
    TcPack *P = new (std::nothrow) TcPack();
    if (!P) return NQS_ENOMEM;
    const int n = M->n, h = M->h, H = sh.Hp, NC = sh.NC, KI = sh.KI, KO = sh.KO, L = M->L;       // H: padded width
    P->Hp = H;
    P->KI = KI; P->KO = KO; P->NC = NC; P->nacc = sh.nacc; P->slot_bytes = sh.slot; P->nslots = sh.nslots; P->split = sh.split;
    const int SP = sh.split;
    P->tm_d3 = (uint32_t)sh.nacc * CN; P->tm_a0 = P->tm_d3 + (uint32_t)KO;
    P->L = smem_layout(H, KO, L, sh.slot, sh.nslots, sh.split);
    const uint32_t slot = sh.slot;
    const uint32_t in_bytes = (uint32_t)HALF * KI * 2, w2_bytes = HALF * 128;
    const std::vector<float> &W1v = M->wm[0], &W3v = M->wm[L];
    auto w1 = [&](int j, int d) { return j < h ? W1v[(size_t)j * n + d] : 0.f; };
    auto p1 = [&](int j, int d) { return j < h ? M->p1[(size_t)j * (n - 2) + d] : 0.f; };
    auto w2 = [&](int j, int k) { return (j < h && k < h) ? M->wm[1][(size_t)j * h + k] : 0.f; };
    auto w3 = [&](int d, int k) { return k < h ? W3v[(size_t)d * h + k] : 0.f; };
    auto p2 = [&](int o, int k) { return k < h ? M->p2[(size_t)o * h + k] : 0.f; };
    auto b1 = [&](int j) { return j < h ? M->bias[0][j] : 0.f; };
    auto c1 = [&](int j) { return j < h ? M->c1[j] : 0.f; };
    auto b2 = [&](int j) { return j < h ? M->bias[1][j] : 0.f; };

    // ---- the per-tile op list (must match the issuer / epilogue loops of eloc_tc_kernel) ----
    int nops = 0;
    auto push_op = [&](uint8_t t, int c) {
        P->optype[nops] = t; P->opchunk[nops] = (uint8_t)c;
        ++nops;
    };
    // The interleaved order issues layer-2 chunk c before the layer-1 chunks > c exist: legal only if no layer-2 chunk has
    // a non-zero weight on a later layer-1 chunk (true for the sorted default degrees, where the masks are prefixes).
    // (The interleaved list has L1S c+1 ahead of L2 c, so a chunk may also read the NEXT layer-1 chunk: with sorted
    // degrees, units on both sides of a chunk boundary can share a degree.)
    if (L == 2)
        for (int c2 = 0; c2 < NC; ++c2)
            for (int r = 0; r < CN; ++r)
                for (int k = (c2 + 2) * CN; k < H; ++k)
                    if (w2(c2 * CN + r, k) != 0.0f) P->seq = 1;
    if (L == 2 && P->seq) {
        for (int c = 0; c < NC; ++c) push_op(T_L1S, c);
        for (int c = 0; c < NC; ++c) { push_op(T_P, c); push_op(T_L2, c); }
    } else if (L == 2) {
        push_op(T_L1S, 0);
        for (int c = 0; c < NC; ++c) {
            if (c + 1 < NC) push_op(T_L1S, c + 1);
            push_op(T_P, c);
            push_op(T_L2, c);
        }
    } else {
        for (int c = 0; c < NC; ++c) { push_op(T_L1I, c); push_op(T_P, c); }
    }
    P->nops = nops;

    std::vector<uint8_t> img[2], res[2];
    res[0].assign((size_t)(1 + SP) * (H / 64) * 1024, 0); res[1] = res[0];
    std::vector<uint2> fills;
    std::vector<uint32_t> sub;
    auto put = [](std::vector<uint8_t> &buf, size_t off, float v) { __half hv = __float2half_rn(v); memcpy(&buf[off], &hv, 2); };
    // part 0: the fp16 rounding of v (all there is in single-pass mode); part 1: the fp16 rounding of what part 0 lost
    auto part_of = [](float v, int part) { const float hi = __half2float(__float2half_rn(v)); return part == 0 ? hi : v - hi; };

    // ---- streamed sub-tiles are appended to the open ring fill (<= slot bytes, in consumption order) ----
    uint32_t fill_start = 0, fill_bytes = 0;
    auto close_fill = [&]() {
        if (fill_bytes == 0) return;
        fills.push_back(make_uint2(fill_start, fill_bytes));
        sub.back() |= SUB_END;
        fill_bytes = 0;
    };
    auto stream_alloc = [&](uint32_t bytes, uint32_t aux) -> uint32_t {
        if (fill_bytes + bytes > slot) close_fill();
        uint32_t w = (aux & 0xFFu) << SUB_AUX_SHIFT;
        if (fill_bytes == 0) { fill_start = (uint32_t)img[0].size(); w |= SUB_NEW; }
        w |= (fill_bytes >> 4) & SUB_OFF_MASK;
        const uint32_t base = fill_start + fill_bytes;
        img[0].resize(img[0].size() + bytes, 0); img[1].resize(img[1].size() + bytes, 0);
        fill_bytes += bytes;
        sub.push_back(w);
        return base;
    };

    // input-layer chunk c (layer 1 or phase hidden): rank r holds units 128 c + 64 r .. + 63.  Masked layer-1 columns
    // are the high ones for sorted degrees; in general the issued K-steps are the prefix up to the last non-zero one.
    auto input_chunk = [&](int c, bool phase) {
        for (int part = 0; part <= SP; ++part) {
            const uint32_t base = stream_alloc(in_bytes, 0);
            int nk = 1;                                         // the accumulator must be overwritten even if all zero
            for (int r = 0; r < 2; ++r)
                for (int rr = 0; rr < HALF; ++rr) {
                    const int j = c * CN + r * HALF + rr;
                    const float bj = phase ? c1(j) : b1(j);
                    const float bj_hi = __half2float(__float2half_rn(bj));
                    for (int k = 0; k < KI; ++k) {
                        float v = 0.f;                          // K index 0, 1: bias (hi, lo) against the constant +1 inputs
                        const int d = k - 2;
                        if (k == 0) v = part == 0 ? bj_hi : 0.f;
                        else if (k == 1) v = part == 0 ? bj - bj_hi : 0.f;
                        else if (phase) { if (d < n - 2) v = part_of(p1(j, d), part); }
                        else if (d < n) v = part_of(w1(j, d), part);
                        put(img[r], base + noswz_offset(rr, k, KI), v);
                        if (v != 0.0f && k / 16 + 1 > nk) nk = k / 16 + 1;
                    }
                }
            sub.back() |= ((uint32_t)nk << SUB_AUX_SHIFT) | (part ? SUB_ACC : 0u);
            P->mma_issued += (long long)nk * CN;
        }
        P->mma_dense += (long long)(KI / 16) * CN;
    };
    // resident P2 tile of phase chunk c: rows 12..15 of the 16-row tile hold the 4 phase outputs -> rank 1, rows 4..7
    auto phase_out_tile = [&](int c) {
        for (int part = 0; part <= SP; ++part)
            for (int o = 0; o < 4; ++o)
                for (int k = 0; k < CN; ++k)
                    put(res[1], (size_t)(c * (1 + SP) + part) * 2048 + (size_t)(k / 64) * 1024 + sw128_offset(4 + o, k % 64),
                        part_of(p2(o, c * CN + k), part));
        P->mma_issued += (1 + 2 * SP) * 8 * 16; P->mma_dense += 8 * 16;
    };
    // layer-2 chunk c2: k-blocks of 64 with any non-zero weight, and inside a block only the non-zero K-steps
    auto l2_chunk = [&](int c2) {
        {   // bias rows of the chunk, one K-step wide: K index 0, 1 = b2 (hi, lo), the rest 0 (A operand = A0's first K-step)
            const uint32_t base = stream_alloc(HALF * 16 * 2, 0);
            for (int r = 0; r < 2; ++r)
                for (int rr = 0; rr < HALF; ++rr) {
                    const float bj = b2(c2 * CN + r * HALF + rr);
                    const float bj_hi = __half2float(__float2half_rn(bj));
                    put(img[r], base + noswz_offset(rr, 0, 16), bj_hi);
                    put(img[r], base + noswz_offset(rr, 1, 16), bj - bj_hi);
                }
            P->mma_issued += CN;
        }
        int nb = 0, need = 0;
        for (int kb = 0; kb < H / 64; ++kb) {
            uint32_t kmask = 0;
            for (int r = 0; r < CN; ++r)
                for (int k = 0; k < 64; ++k)
                    if (w2(c2 * CN + r, kb * 64 + k) != 0.0f) kmask |= 1u << (k / 16);
            P->mma_dense += 4 * CN;
            if (!kmask) continue;                                        // exact: an all-zero block adds 0
            // single pass: A1[kb] . W2^T.  Split: A1hi[kb] . W2hi^T + A1lo[kb] . W2hi^T + A1hi[kb] . W2lo^T — two
            // streamed blocks (weight parts); the lo activations live H/64 k-blocks after the hi ones
            // (the hi weight block is streamed once and used against both activation parts: flag SUB_ACC)
            const int npass = SP ? 2 : 1;
            for (int ps = 0; ps < npass; ++ps) {
                const int a_kb = kb, wpart = ps;
                const uint32_t base = stream_alloc(w2_bytes, (uint32_t)a_kb | (kmask << 4));
                if (SP && ps == 0) sub.back() |= SUB_ACC;
                for (int r = 0; r < 2; ++r)
                    for (int rr = 0; rr < HALF; ++rr)
                        for (int k = 0; k < 64; ++k)
                            put(img[r], base + sw128_offset(rr, k), part_of(w2(c2 * CN + r * HALF + rr, kb * 64 + k), wpart));
                P->mma_issued += (long long)__builtin_popcount(kmask) * CN * ((SP && ps == 0) ? 2 : 1);
                ++nb;
            }
            need = kb / 2;
        }
        P->nblk[c2] = (uint8_t)nb; P->l2need[c2] = (uint8_t)need;
    };
    // streamed layer-3 tile of hidden chunk c: N = KO - n_lo output rows (rows below the first non-zero one receive
    // exactly 0 from this chunk), rank r holds rows n_lo + r N/2 .. ; two K-blocks of N/2 rows x 128 B
    auto w3_tile = [&](int c) {
        int row_lo = KO;
        for (int d = 0; d < n; ++d)
            for (int k = 0; k < CN; ++k)
                if (w3(d, c * CN + k) != 0.0f && d < row_lo) row_lo = d;
        const int n_lo = row_lo >= KO ? KO - 16 : (row_lo / 16) * 16;
        const int N = KO - n_lo, Nh = N / 2;
        const uint32_t tile_bytes = (uint32_t)2 * Nh * 128;                   // split: the lo-part tile follows the hi-part tile
        const uint32_t base = stream_alloc(tile_bytes * (1 + SP), (uint32_t)(n_lo / 16));
        for (int part = 0; part <= SP; ++part)
            for (int r = 0; r < 2; ++r)
                for (int rr = 0; rr < Nh; ++rr) {
                    const int d = n_lo + r * Nh + rr;
                    if (d >= n) continue;
                    for (int k = 0; k < CN; ++k)
                        put(img[r], base + part * tile_bytes + (size_t)(k / 64) * Nh * 128 + sw128_offset(rr, k % 64),
                            part_of(w3(d, c * CN + k), part));
                }
        P->mma_issued += (long long)(1 + 2 * SP) * 8 * N; P->mma_dense += (long long)8 * KO;
    };
    auto emit_op = [&](int j) {
        const int c = P->opchunk[j];
        switch (P->optype[j]) {
            case T_L1S: case T_L1I: input_chunk(c, false); break;
            case T_P: input_chunk(c, true); phase_out_tile(c); break;
            default: l2_chunk(c); break;
        }
    };
    auto emit_consumer = [&](int j) {
        if (P->optype[j] == T_L2 || P->optype[j] == T_L1I) w3_tile(P->opchunk[j]);
    };
    const int lag = sh.nacc - 1;
    for (int j = 0; j < nops; ++j) { emit_op(j); if (j >= lag) emit_consumer(j - lag); }
    for (int m = lag; m >= 1; --m) if (nops >= m) emit_consumer(nops - m);
    close_fill();
    // ---- where the issuer waits for chunk epilogues that have no consumer MMA (layer-1 chunks written to A1): before
    // the accumulator's next producer or the first layer-2 op that reads the chunk, whichever is issued first ----
    if (L == 2) P->l2need[NC - 1] = (uint8_t)(NC - 1);          // every layer-1 epilogue is waited for inside its own tile
    {
        int pending[3] = {-1, -1, -1};
        int l1s_op[MAX_NC] = {0};
        for (int j = 0; j < nops; ++j) if (P->optype[j] == T_L1S) l1s_op[P->opchunk[j]] = j;
        for (int j = 0; j < nops; ++j)                           // every layer-1 chunk a layer-2 op reads is issued before it
            if (P->optype[j] == T_L2)
                for (int cn = 0; cn <= P->l2need[P->opchunk[j]]; ++cn)
                    if (l1s_op[cn] > j) { delete P; return NQS_EUNSUPPORTED; }
        auto consumed = [&](int j) { if (P->optype[j] != T_L1S && pending[j % sh.nacc] == j) pending[j % sh.nacc] = -1; };
        for (int j = 0; j < nops; ++j) {
            const int a = j % sh.nacc;
            uint8_t pw = 0;
            if (pending[a] >= 0) { pw |= (uint8_t)(1u << a); pending[a] = -1; }
            if (P->optype[j] == T_L2)
                for (int cn = 0; cn <= P->l2need[P->opchunk[j]]; ++cn) {
                    const int jo = l1s_op[cn], ao = jo % sh.nacc;
                    if (pending[ao] == jo) { pw |= (uint8_t)(1u << ao); pending[ao] = -1; }
                }
            P->prewait[j] = pw;
            pending[a] = j;
            if (j >= lag) consumed(j - lag);
        }
        for (int m = lag; m >= 1; --m) if (nops >= m) consumed(nops - m);
        if (pending[0] >= 0 || pending[1] >= 0 || pending[2] >= 0) { delete P; return NQS_EUNSUPPORTED; }
        for (int a = 0; a < sh.nacc; ++a) {
            int cnt = 0;
            for (int j = a; j < nops; j += sh.nacc) ++cnt;
            if (cnt & 1) P->cntmask |= 1u << a;
        }
    }
    P->nsub = (int)sub.size(); P->nfills = (int)fills.size();
    P->res_bytes = (uint32_t)res[0].size();
    if (P->nsub > MAX_SUB) { delete P; return NQS_EUNSUPPORTED; }
    memcpy(P->sub, sub.data(), sub.size() * 4);
    P->img_stride = (uint32_t)((img[0].size() + 255) & ~(size_t)255);

    // biases left to the final epilogue: [b3 (KO) | c2]
    std::vector<float> bias((size_t)KO + 4, 0.f);
    for (int d = 0; d < n; ++d) bias[d] = M->bias[L][d];
    for (int o = 0; o < 4; ++o) bias[KO + o] = M->c2[o];

    std::vector<uint8_t> wboth((size_t)2 * P->img_stride, 0), rboth((size_t)2 * P->res_bytes, 0);
    for (int r = 0; r < 2; ++r) {
        memcpy(&wboth[(size_t)r * P->img_stride], img[r].data(), img[r].size());
        memcpy(&rboth[(size_t)r * P->res_bytes], res[r].data(), res[r].size());
    }
    int dev = 0; cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&P->sms, cudaDevAttrMultiProcessorCount, dev);
    auto up = [](void **dst, const void *src, size_t bytes) {
        return cudaMalloc(dst, bytes ? bytes : 16) == cudaSuccess && (bytes == 0 || cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice) == cudaSuccess);
    };
    const bool ok = up(&P->d_wimg, wboth.data(), wboth.size()) && up(&P->d_fills, fills.data(), fills.size() * sizeof(uint2)) &&
                    up(&P->d_res, rboth.data(), rboth.size()) && up(&P->d_bias, bias.data(), bias.size() * 4);
    if (!ok) {
        cudaGetLastError();
        cudaFree(P->d_wimg); cudaFree(P->d_fills); cudaFree(P->d_res); cudaFree(P->d_bias);
        delete P;
        return NQS_ECUDA;
    }
    M->tc = P;
    return NQS_OK;
}

void tc_pack_free(const nqs_made *M) {
    if (!M->tc) return;
    TcPack *P = M->tc;
    cudaFree(P->d_wimg); cudaFree(P->d_fills); cudaFree(P->d_res); cudaFree(P->d_bias);
    if (P->d_fpos) cudaFree(P->d_fpos);
    if (P->d_epart) cudaFree(P->d_epart);
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
    p.n = M->n; p.H = P->Hp; p.NC = P->NC; p.KI = P->KI; p.KO = P->KO; p.L = M->L; p.nacc = P->nacc; p.nops = P->nops; p.split = P->split; p.seq = P->seq;
    p.tm_d3 = P->tm_d3; p.tm_a0 = P->tm_a0;
    p.wimg = (const uint8_t *)P->d_wimg; p.img_stride = P->img_stride;
    p.fills = (const uint2 *)P->d_fills; p.nfills = P->nfills;
    memcpy(p.sub, P->sub, sizeof(p.sub)); memcpy(p.nblk, P->nblk, sizeof(p.nblk));
    memcpy(p.optype, P->optype, sizeof(p.optype)); memcpy(p.opchunk, P->opchunk, sizeof(p.opchunk));
    memcpy(p.prewait, P->prewait, sizeof(p.prewait)); p.cntmask = P->cntmask;
    p.resimg = (const uint8_t *)P->d_res; p.res_bytes = P->res_bytes;
    p.slot_bytes = P->slot_bytes; p.nslots = P->nslots;
    p.nprod = P->nslots < NPROD ? P->nslots : NPROD;
    p.bias = (const float *)P->d_bias;
    p.n_up = M->dev.n_up; p.n_down = M->dev.n_down; p.spin_lo = M->dev.spin_lo; p.spin_hi = M->dev.spin_hi;
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


template <int NC, int L, int NACC, bool SPLIT, bool SEQ>
static int launch_inst(const TcParams &p, int grid, uint32_t smem_bytes, cudaStream_t st) {
    using S = Sched<NC, L, NACC, SEQ>;
    if (p.nops != S::NOPS) return NQS_EUNSUPPORTED;
    for (int j = 0; j < S::NOPS; ++j)                        // the host-packed op list must be the compiled schedule
        if (p.optype[j] != S::type(j) || p.opchunk[j] != S::chunk(j)) return NQS_EUNSUPPORTED;
    // the attribute is per device and per kernel; setting it is a cheap host call, so no process-wide cache
    if (cudaFuncSetAttribute(eloc_tc_kernel<NC, L, NACC, SPLIT, SEQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes) != cudaSuccess) {
        cudaGetLastError();
        return NQS_ECUDA;
    }
    eloc_tc_kernel<NC, L, NACC, SPLIT, SEQ><<<grid, NTHREADS, smem_bytes, st>>>(p);
    return NQS_OK;
}

static int launch_chain(const TcPack *P, TcParams &p, long long ntiles, cudaStream_t st) {
    const long long npairs = (ntiles + 1) / 2;
    const long long ncl_max = P->sms / 2;
    const int grid = 2 * (int)(npairs < ncl_max ? npairs : ncl_max);
    int rc = NQS_EUNSUPPORTED;
    // hidden <= 256 runs in split precision (tc_shape), wider nets in a single fp16 pass
#define TC_CASE(NC_, L_, NA_, SP_) case (NC_ * 16 + L_ * 4 + NA_): \
        rc = (L_ == 2 && p.seq) ? launch_inst<NC_, L_, NA_, SP_, (L_ == 2)>(p, grid, P->L.total, st) \
                                : launch_inst<NC_, L_, NA_, SP_, false>(p, grid, P->L.total, st); break;
    if ((p.split != 0) != (p.NC <= 2)) return NQS_EUNSUPPORTED;
    switch (p.NC * 16 + p.L * 4 + p.nacc) {
        TC_CASE(1, 1, 2, true) TC_CASE(2, 1, 2, true) TC_CASE(3, 1, 2, false) TC_CASE(4, 1, 2, false)
        TC_CASE(1, 2, 2, true) TC_CASE(2, 2, 2, true) TC_CASE(3, 2, 2, false) TC_CASE(4, 2, 2, false)
        TC_CASE(1, 1, 3, true) TC_CASE(2, 1, 3, true) TC_CASE(3, 1, 3, false) TC_CASE(4, 1, 3, false)
        TC_CASE(1, 2, 3, true) TC_CASE(2, 2, 3, true) TC_CASE(3, 2, 3, false) TC_CASE(4, 2, 3, false)
        default: break;
    }
#undef TC_CASE
    if (rc) return rc;
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
    return launch_chain(P, p, (B + TILE_M - 1) / TILE_M, st);
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
    TcParams p{};
    fill_common(M, p);
    p.mode = 1; p.xpos = (const ulonglong2 *)P->d_xpos; p.B = B; p.fpos = (const ulonglong2 *)P->d_fpos; p.x = x;
    p.hm = hm; p.base = base; p.max_ratio_bits = max_ratio_bits;
    p.g_begin = hm.has_diag ? 1 : 0;
    const long long nsb = (B + TILE_M - 1) / TILE_M;
    const long long Gnd = hm.G - p.g_begin;
    const long long ntiles = nsb * Gnd;
    // Partial-sum slots (see the flush in the kernel): walk the kernel's own static schedule -- cluster k owns tile pairs
    // [npairs k / ncl, npairs (k+1) / ncl) -- and take the largest number of clusters that share one sample block.
    int eslots = 0;
    if (ntiles > 0) {
        const long long npairs = (ntiles + 1) / 2, ncl_max = P->sms / 2, ncl = npairs < ncl_max ? npairs : ncl_max;
        long long cur_sb = -1, cnt = 0, most = 0;
        for (long long k = 0; k < ncl; ++k) {
            const long long t_lo = 2 * (npairs * k / ncl), t_hi = std::min(2 * (npairs * (k + 1) / ncl), ntiles);
            if (t_hi <= t_lo) continue;
            const long long sb_lo = t_lo / Gnd, sb_hi = (t_hi - 1) / Gnd;
            cnt = (sb_lo == cur_sb) ? cnt + 1 : 1;                 // clusters on block sb_lo so far
            most = std::max(most, cnt);
            if (sb_hi != sb_lo) cnt = 1;                           // this cluster is the first on block sb_hi (blocks between are its own)
            cur_sb = sb_hi;
        }
        eslots = (int)(2 * most);
        const size_t bytes = sizeof(float2) * (size_t)nsb * eslots * TILE_M;
        if ((rc = ensure(&P->d_epart, &P->epart_cap, bytes))) return rc;
        if (cudaMemsetAsync(P->d_epart, 0, bytes, st) != cudaSuccess) { cudaGetLastError(); return NQS_ECUDA; }
        p.epart = (float2 *)P->d_epart; p.eslots = eslots;
        if ((rc = launch_chain(P, p, ntiles, st))) return rc;
    }
    eloc_finish_kernel<<<(unsigned)((B + 255) / 256), 256, 0, st>>>(hm, x, B, (const float2 *)P->d_epart, eslots, eloc);
    ++g_launch_count;
    return cudaGetLastError() == cudaSuccess ? NQS_OK : NQS_ECUDA;
}

