// kernel.cuh -- the persistent, warp-specialised sm_100a kernel of the CTA-pipelined chained GEMM.
//
// One launch runs layers [layer_begin, layer_end) of the chain  A^l = bf16(act(A^{l-1} . W_l)).
// CTA_PIPELINED launches it once over all layers; SEQUENTIAL / MICROBATCH launch it once per
// layer (and per row chunk) with the protocol's waiting switched off.
//
// Orientation ("weights fill the 128-row MMA slot"): per work unit the tensor
// core computes  D[n, m] = sum_k W_l[n, k] * A^{l-1}[m, k]  with
//     A operand = W tile      128 weight rows (n) x 64 k, K-major, 128B swizzle   (16 KB)
//     B operand = activation  tile_m tokens (m)   x 64 k, K-major, 128B swizzle   (tile_m * 128 B)
//     D         = TMEM, lane = n (128 lanes), column = m (tile_m fp32 columns), a ring of accumulators
// so that a decode-sized batch (M = 16) costs a 128 x 16 MMA instead of a padded 128 x 128 one and
// every weight byte is loaded exactly once.  With n_sub = 2 a unit covers 256 weight rows (two
// 128-row MMAs per K step that share the activation tile in shared memory), which halves the
// activation bytes pulled from L2 per weight byte -- what bounds the kernel once M >= 128.
//
// Work units come from a per-layer UNIT TABLE written by the host (mlp_pipe.cu: resolve): ticket t
// of layer l is table_l[t].  Two kinds: an MMA unit (tile, K-slice [kb0, kb1)) and a REDUCE unit
// (tile, token columns [c0, c1)) that sums the split-K partials of a tile in fixed slice order.  A
// unit only ever depends on units with a lower ticket of its own layer (reduce after its slices) or
// on units of the layer before.
//
// Warp roles (protocol hidden in the scheduler and store warps of a
// warp-specialised persistent kernel):
//     warp 0  scheduler     global atomic ticket -> unit table -> smem ring (broadcast), drawn late; fast-path look
//                            at the unit's ready counters; in work-queue mode: pops the unit from the queue  [step a1]
//     warp 1  W loader      TMA loads of weight tiles; never waits on a flag, so W_{l+1} is
//                            prefetched up to the ring depth before A^l exists (32 lanes converged, one elected issuer)
//     warp 2  A loader      consumer prologue: polls the (M-block, K-slice) ready counters (ld.relaxed.gpu + one
//                            fence.acq_rel.gpu, or ld.acquire.gpu), then TMA-loads the activation tile [step a5]
//                            (32 lanes converged, one elected lane issues the TMA)
//     warp 3  MMA issuer    tcgen05.mma into TMEM (32 lanes converged, one elected lane issues: the issue loop paces
//                            the tensor pipe, see the role); owns TMEM alloc / dealloc       [a2, a6]
//     warps 4-7 epilogue    tcgen05.ld -> act -> bf16 -> transposed store, or fp32 split-K partial (+ gather by the
//                            last arriver), or a reduce unit; then producer epilogue: fence + red.release.gpu
//                            publish (+ scoreboard / queue push in work-queue mode)          [a3, a4, a7, a8]
#pragma once
#include <cuda_bf16.h>

#include "ptx.cuh"

namespace mlp {

constexpr int kMaxLayers = 8;
constexpr int kTileN = 128;  // weight rows per tile (UMMA M)
constexpr int kTileK = 64;   // bf16 per smem row = 128 B = one swizzle span
constexpr int kUmmaK = 16;
constexpr int kMaxStages = 16;
constexpr int kSchedSlots = 4;
constexpr int kThreads = 256;
constexpr int kEpiThreads = 128;
constexpr int kWTileBytes = kTileN * kTileK * 2;
constexpr int kCtrlBytes = 1024;
constexpr int kUnitTrace = 12;
constexpr int kMaxAccStages = 8;
constexpr int kGather = 7;  // split-K partials fetched per round trip by the reducer
constexpr int kStageTokens = 32;                            // tokens per epilogue staging buffer
constexpr int kStageBufBytes = kStageTokens * kTileN * 2;   // [32 tokens][128 features] bf16
constexpr int kStageBytes = 2 * kStageBufBytes;             // double buffered
constexpr int kUnitMma = 0, kUnitReduce = 1;
constexpr int kReduceNone = 0, kReduceLastArriver = 1, kReduceUnits = 2;

// One entry of a layer's unit table = one ticket.
struct UnitDesc {
    uint16_t tile;  // m_blk * n_blks + n_blk
    uint8_t kind;   // kUnitMma | kUnitReduce
    uint8_t ks;     // K-slice index (MMA unit)
    uint16_t a, b;  // MMA unit: K-blocks [a, b); reduce unit: token columns [a, b) of the tile
};
static_assert(sizeof(UnitDesc) == 8, "UnitDesc is read as one 8-byte word");

constexpr int kActNone = 0, kActRelu = 1, kActGeluTanh = 2;
constexpr float kGelu0 = 0.7978845608028654f, kGelu1 = 0.7978845608028654f * 0.044715f;  // sqrt(2/pi), sqrt(2/pi) * 0.044715
constexpr uint32_t kFlagTileMajor = 0x1u, kFlagDebugDelay = 0x2u, kFlagDebugReverse = 0x4u, kFlagNoEvictFirst = 0x8u;
// measurement knobs (include/mlp_pipe.h MLP_FLAG_EXP_*): each removes or replaces one protocol ingredient
constexpr uint32_t kFlagExpNoAcquireFence = 0x10u, kFlagExpNoProxyFence = 0x20u, kFlagAcquireLoads = 0x40u,
                   kFlagExpNoFastPath = 0x80u, kFlagExpNoPreissue = 0x100u;
constexpr uint32_t kFlagWorkQueue = 0x1000u;  // consumers pop ready units from a work queue instead of polling ready counters
constexpr uint32_t kFlagPdl = 0x800u;  // SEQUENTIAL: layer l+1 is launched as a programmatic dependent of layer l
constexpr uint32_t kFlagDebugDropPublish = 0x4000u;  // test hook: the producer of tile 0 of the launch's first layer never publishes
constexpr uint32_t kStatusFlagTimeout = 1u;

struct LayerParams {
    int K, N;
    int kb_total;  // ceil(K / 64)
    int n_blks;    // ceil(N / (128 * n_sub))
    int split;     // split of the contraction per output tile
    int units;     // entries of the unit table (MMA units + reduce units)
    int ticket_inc;  // what one launch adds to the ticket counter: units + CTAs arriving from the layer before
    int ticket_off;  // unit index of the first atomically drawn ticket (= units handed out statically)
    int act;       // activation on this layer's output
    int publish;   // 1 if a later layer consumes this layer's output
    int static_sp;    // > 0: tickets t < grid of this layer are MMA units (tile t / static_sp, slice t % static_sp, equal
                      // slices) -- lets a CTA decode its static first unit without reading the table
    int reduce_mode;  // kReduceNone (split == 1) | kReduceLastArriver | kReduceUnits
    int ready_inc;    // what one run adds to a tile's ready counter (1, or its number of reduce units)
    __nv_bfloat16* out;  // [M x N] row-major
    float* ws;           // split-K partials [tile][split][n_sub][tile_m / 4][128][4]
    uint32_t* ticket;    // 1 monotone counter
    uint32_t* arrive;    // [tiles] monotone split-K arrival counters
    uint32_t* ready;     // [tiles] monotone ready counters, tile = m_blk * n_blks + n_blk
    const UnitDesc* table;  // [units] ticket -> unit
    // ---- the paper's literal protocol, MLP_FLAG_WORKQUEUE: dependency array -> scoreboard -> work queue.
    // A GROUP of this layer = its units with the same (M-block, K-slice): they depend on the same producer tiles.
    int use_queue;               // 1: tickets of this layer index its work queue (unit order = order in which groups become ready)
    int group_units;             // units per group (= N-tiles per M-block)
    uint32_t* scoreboard;        // [groups] monotone: += 1 per finished producer tile the group depends on
    uint32_t* qtail;             // 1 monotone counter: next free queue slot
    uint32_t* queue;             // [units] slot = (epoch tag << 16) | table index
    const uint16_t* dep_count;   // [groups] producer tiles a group depends on
    const uint16_t* qorder;      // [groups][group_units] table indices of a group's units
    const uint16_t* dep_off;     // [tiles of the layer BEFORE + 1] CSR offsets into dep_list: "dependency array" of a producer tile
    const uint16_t* dep_list;    // groups of THIS layer that depend on that producer tile
};

struct CtaStats {
    unsigned long long stall_cycles;
    unsigned long long polls;
    unsigned long long cycles;
    unsigned long long ts[8];  // globaltimer ns: 0 start, 1 setup done, 2 first ticket, 3 first W TMA issued,
                               // 4 first stage landed, 5 first accumulator ready, 6 first unit stored, 7 exit
    unsigned long long wait[8];  // SM cycles: 0 W loader blocked on a free stage, 1 reducer summing partials,
                                 // 2 MMA blocked on operands, 3 MMA blocked on a free accumulator, 4 epilogue
                                 // blocked on an accumulator, 5 reduce unit blocked on its tile's arrival counter,
                                 // 6 storing split-K partials, 7 direct epilogue
    uint32_t units[kMaxLayers];
    unsigned long long unit_ts[kUnitTrace][4];  // per executed unit: W loader start, W loader done issuing,
                                                // accumulator complete, epilogue done (globaltimer ns)
    uint32_t unit_id[kUnitTrace];               // layer << 28 | tile << 8 | ks
};

struct KernelParams {
    CUtensorMap tm_w[kMaxLayers];
    CUtensorMap tm_a[kMaxLayers];  // input activations of layer l: X (l = 0) or H_l
    LayerParams layer[kMaxLayers];
    int layer_begin, layer_end;
    int m_off, m_end;  // token rows [m_off, m_end) of this launch
    int tile_m, m_blks;
    int n_sub;          // 128-row MMAs per unit and K step (1 or 2): a unit covers 128 * n_sub weight rows
    int stages;         // weight ring depth
    int a_stages;       // activation ring depth
    int acc_stages;     // TMEM accumulators in the ring
    int claim_ahead;    // the scheduler draws the next ticket when the weight loader has this many K-blocks left
    int w_group;        // weight K-blocks requested back to back
    int producer_ctas;  // CTAs with blockIdx.x < producer_ctas start at layer_begin, the rest one layer later
    int wait_flags;     // consumer prologue on/off
    int pair;           // 1: CTA pairs (cluster of 2, tcgen05 cta_group::2): a pair executes one unit of 256 weight rows, each
                        // CTA loading its 128 rows and HALF of the activation tile; the leader (rank 0) schedules and issues
    int wait_first;     // 1: the launch's FIRST layer is a consumer too -- its producer runs in another launch on another
                        // stream (MLP_FLAG_TWO_KERNEL) and publishes the same ready counters
    int pdl_wait;       // 1: launched as a programmatic dependent; the activation loader waits for the grid before
    uint32_t flags;
    unsigned long long* epoch_counter;  // += 1 per exiting CTA; epoch = value / gridDim.x
    uint32_t* status;
    uint32_t* status_host;  // the same word mirrored in pinned host memory (written on expiry only): mlp_pipe_run reads it for free
    unsigned long long timeout_ns;
    CtaStats* stats;
};

struct UnitInfo {
    int layer, m_blk, n_blk, ks, kb0, kb1, valid, tile;
    int acquired;  // 1: the scheduler has already seen (and acquired) every counter this unit depends on
    int kind;      // kUnitMma | kUnitReduce (then kb0, kb1 = token columns)
    int pad_[2];
};

template <int act>
__device__ __forceinline__ float act_apply(float x) {
    if (act == kActRelu) return x > 0.0f ? x : 0.0f;
    if (act == kActGeluTanh) {
        // g(x) = 0.5 x (1 + tanh(sqrt(2/pi) (x + 0.044715 x^3))) as mul, fma, mul, MUFU, mul, fma; kGelu1 = sqrt(2/pi) * 0.044715
        const float u = x * fmaf(x * x, kGelu1, kGelu0);
        float t;
        asm("tanh.approx.f32 %0, %1;" : "=f"(t) : "f"(u));
        const float hx = 0.5f * x;
        return fmaf(hx, t, hx);
    }
    return x;
}

// Two GeLUs at once on the packed fp32 pipe (mul.f32x2 / fma.rn.f32x2: one issue slot per pair), the same operations in
// the same order as act_apply<kActGeluTanh> lane by lane, so the result is bit-identical to it: the epilogue warps (one
// per sub-partition) are issue-bound at large token tiles, and the arithmetic of the activation is most of their slots.
__device__ __forceinline__ void gelu_tanh_x2(float xa, float xb, float& ya, float& yb) {
    uint64_t x, c0, c1, h, u, t, y;
    float ua, ub, ta, tb;
    asm("mov.b64 %0, {%1, %2};" : "=l"(x) : "f"(xa), "f"(xb));
    asm("mov.b64 %0, {%1, %1};" : "=l"(c0) : "f"(kGelu0));
    asm("mov.b64 %0, {%1, %1};" : "=l"(c1) : "f"(kGelu1));
    asm("mov.b64 %0, {%1, %1};" : "=l"(h) : "f"(0.5f));
    asm("{\n\t.reg .b64 x2, p;\n\t"
        "mul.f32x2 x2, %1, %1;\n\t"
        "fma.rn.f32x2 p, x2, %2, %3;\n\t"
        "mul.f32x2 %0, %1, p;\n\t}"
        : "=l"(u) : "l"(x), "l"(c1), "l"(c0));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(ua), "=f"(ub) : "l"(u));
    asm("tanh.approx.f32 %0, %1;" : "=f"(ta) : "f"(ua));
    asm("tanh.approx.f32 %0, %1;" : "=f"(tb) : "f"(ub));
    asm("mov.b64 %0, {%1, %2};" : "=l"(t) : "f"(ta), "f"(tb));
    asm("{\n\t.reg .b64 hx;\n\t"
        "mul.f32x2 hx, %1, %2;\n\t"
        "fma.rn.f32x2 %0, hx, %3, hx;\n\t}"
        : "=l"(y) : "l"(x), "l"(h), "l"(t));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(ya), "=f"(yb) : "l"(y));
}

__device__ __forceinline__ float ld_cg_f32(const float* p) {
    float v;
    asm volatile("ld.global.cg.f32 %0, [%1];" : "=f"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void mbar_wait_timed(uint32_t bar, uint32_t parity, unsigned long long& acc) {
    if (mbar_probe(bar, parity)) return;
    const long long t0 = clock64();
    mbar_wait(bar, parity);
    acc += static_cast<unsigned long long>(clock64() - t0);
}

__device__ __forceinline__ void st_cg_f32(float* p, float v) {
    asm volatile("st.global.cg.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory");
}

__device__ __forceinline__ void st_cg_f32x4(float* p, float a, float b, float c, float d) {
    asm volatile("st.global.cg.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
__device__ __forceinline__ float4 ld_cg_f32x4(const float* p) {
    float4 v;
    asm volatile("ld.global.cg.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_shared_b16(uint32_t addr, uint16_t v) {
    asm volatile("st.shared.b16 [%0], %1;" ::"r"(addr), "h"(v) : "memory");
}
__device__ __forceinline__ uint4 ld_shared_v4(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
    return v;
}

// Epilogue output path (steps a3 / a7).  The accumulator is feature-major (TMEM lane = output
// feature n, column = token m) while the output is token-major, so a chunk of up to 32 token columns
// of one 128-feature block is transposed through a shared-memory staging buffer: every thread
// converts its feature's values (act, RNE to bf16) and writes them at stage[token][feature]; after a
// barrier among the 128 epilogue threads the buffer leaves as 16-byte pieces, a warp storing two
// complete 256-byte output rows per instruction.  Two buffers alternate (`parity`), so one barrier
// per chunk suffices: a buffer is rewritten only after the barrier of the chunk in between.
template <int kCols, int kAct>
__device__ __forceinline__ void stage_cols(const uint32_t (&f)[kCols], uint32_t buf, int r) {
    // the activation is a compile-time choice here: a run-time switch per element would serialise the
    // 32 independent columns behind one another's MUFU latency
    if constexpr (kAct == kActGeluTanh) {
#pragma unroll
        for (int j = 0; j < kCols; j += 2) {
            float ya, yb;
            gelu_tanh_x2(__uint_as_float(f[j]), __uint_as_float(f[j + 1]), ya, yb);
            st_shared_b16(buf + static_cast<uint32_t>(j * kTileN + r) * 2u, __bfloat16_as_ushort(__float2bfloat16_rn(ya)));
            st_shared_b16(buf + static_cast<uint32_t>((j + 1) * kTileN + r) * 2u, __bfloat16_as_ushort(__float2bfloat16_rn(yb)));
        }
    } else {
#pragma unroll
        for (int j = 0; j < kCols; ++j)
            st_shared_b16(buf + static_cast<uint32_t>(j * kTileN + r) * 2u, __bfloat16_as_ushort(__float2bfloat16_rn(act_apply<kAct>(__uint_as_float(f[j])))));
    }
}

template <int kCols>
__device__ __forceinline__ void emit_cols(const uint32_t (&f)[kCols], uint32_t stage_s, uint32_t& parity, int r,
                                          __nv_bfloat16* out, size_t ld, int n_base, int N, int m_first, int m_end,
                                          int act) {
    const uint32_t buf = stage_s + (parity & 1u) * kStageBufBytes;
    parity ^= 1u;
    if (act == kActGeluTanh) stage_cols<kCols, kActGeluTanh>(f, buf, r);
    else if (act == kActRelu) stage_cols<kCols, kActRelu>(f, buf, r);
    else stage_cols<kCols, kActNone>(f, buf, r);
    bar_sync(1, kEpiThreads);
    // all shared-memory reads first, then all global stores: the pieces are independent, one exposed latency instead of one per piece
    uint4 v[kCols * 16 / kEpiThreads];
#pragma unroll
    for (int p = 0; p < kCols * 16 / kEpiThreads; ++p) {
        const int piece = p * kEpiThreads + r;  // 16 pieces of 8 features per token row
        v[p] = ld_shared_v4(buf + static_cast<uint32_t>((piece >> 4) * kTileN + (piece & 15) * 8) * 2u);
    }
#pragma unroll
    for (int p = 0; p < kCols * 16 / kEpiThreads; ++p) {
        const int piece = p * kEpiThreads + r;
        const int j = piece >> 4, q = piece & 15;
        const int m = m_first + j, n = n_base + q * 8;
        if (m < m_end && n < N) *reinterpret_cast<uint4*>(out + static_cast<size_t>(m) * ld + n) = v[p];
    }
}

// Sum 16 token columns [c, c+16) of feature r over the `split` partials of one 128-row block, always in
// slice order 0..split-1 (the rounding never depends on who reduces, nor on arrival order).  `blk` points
// at slice 0; slices are `ks_stride` floats apart; layout inside a slice block: [column / 4][128][4].
__device__ __forceinline__ void gather16(const float* blk, int split, size_t ks_stride, int c, int r, float (&sum)[16]) {
    const float* p0 = blk + (static_cast<size_t>(c >> 2) * kTileN + r) * 4;
    for (int ks = 0; ks < split; ks += kGather) {
        float4 t[kGather][4];
#pragma unroll
        for (int q = 0; q < kGather; ++q)
            if (ks + q < split) {
#pragma unroll
                for (int g = 0; g < 4; ++g) t[q][g] = ld_cg_f32x4(p0 + (ks + q) * ks_stride + static_cast<size_t>(g) * kTileN * 4);
            }
#pragma unroll
        for (int q = 0; q < kGather; ++q)
            if (ks + q < split) {
                if (ks + q == 0) {
#pragma unroll
                    for (int g = 0; g < 4; ++g) {
                        sum[4 * g] = t[q][g].x; sum[4 * g + 1] = t[q][g].y; sum[4 * g + 2] = t[q][g].z; sum[4 * g + 3] = t[q][g].w;
                    }
                } else {
#pragma unroll
                    for (int g = 0; g < 4; ++g) {
                        sum[4 * g] += t[q][g].x; sum[4 * g + 1] += t[q][g].y; sum[4 * g + 2] += t[q][g].z; sum[4 * g + 3] += t[q][g].w;
                    }
                }
            }
    }
}

template <int kC>
__device__ __forceinline__ void tmem_ld_cols(uint32_t taddr, uint32_t (&v)[kC]);
template <>
__device__ __forceinline__ void tmem_ld_cols<16>(uint32_t taddr, uint32_t (&v)[16]) { tmem_ld16(taddr, v); }
template <>
__device__ __forceinline__ void tmem_ld_cols<32>(uint32_t taddr, uint32_t (&v)[32]) { tmem_ld32(taddr, v); }

// Context of one epilogue thread's output path.
struct EmitCtx {
    uint32_t stage_s;
    int r;
    __nv_bfloat16* out;
    size_t ld;
    int n_first, N, m0, m_end, act, tile_m;
};

__device__ __forceinline__ void release_acc(uint32_t bar) {  // bar & 1: pair mode, arrive on the LEADER's barrier at this offset
    tc_fence_before();
    if (bar & 1u) mbar_arrive_cluster((bar & ~1u) & kPeerBitMask);
    else mbar_arrive(bar);
}

template <int kC>
__device__ __forceinline__ void emit_chunk(const uint32_t (&v)[kC], int cc, const EmitCtx& e, uint32_t& parity) {
    const int rr = cc >= e.tile_m ? 1 : 0, c = cc - rr * e.tile_m;
    emit_cols<kC>(v, e.stage_s, parity, e.r, e.out, e.ld, e.n_first + rr * kTileN, e.N, e.m0 + c, e.m_end, e.act);
}

template <int kC>
__device__ __forceinline__ void store_chunk(const uint32_t (&v)[kC], int cc, float* wsp) {
#pragma unroll
    for (int g = 0; g < kC / 4; ++g)
        st_cg_f32x4(wsp + static_cast<size_t>((cc >> 2) + g) * kTileN * 4, __uint_as_float(v[4 * g]), __uint_as_float(v[4 * g + 1]),
                    __uint_as_float(v[4 * g + 2]), __uint_as_float(v[4 * g + 3]));
}

// ---- direct epilogue in the MMA-fragment shape (steps a3 / a7).  The accumulator is feature-major (TMEM lane = feature,
// column = token), the output token-major.  Read with tcgen05.ld.16x256b a thread holds, for one feature, PAIRS of
// adjacent tokens -- exactly the register shape stmatrix.trans wants: act + cvt.rn.bf16x2 on the pair, then ONE
// stmatrix.x4.trans per 16 lanes x 16 tokens writes 16 token rows of 16 features each into the staging buffer (the
// transpose is done by the store unit, 512 bytes per instruction instead of 64 for a 2-byte st.shared per element: the
// epilogue warps were bound by the number of load/store-unit instructions).  Token rows are kFragPitch bytes apart (256 + 16:
// the 8 rows of a matrix then fall into different banks).  Leaves as 16-byte pieces exactly like emit_cols.
constexpr uint32_t kFragPitch = kTileN * 2 + 16;
static_assert(16 * kFragPitch <= kStageBufBytes, "16 token rows must fit a staging buffer");

template <int kAct>
__device__ __forceinline__ uint32_t frag_pack(uint32_t a, uint32_t b) {
    float ya, yb;
    if constexpr (kAct == kActGeluTanh) {
        gelu_tanh_x2(__uint_as_float(a), __uint_as_float(b), ya, yb);
    } else {
        ya = act_apply<kAct>(__uint_as_float(a));
        yb = act_apply<kAct>(__uint_as_float(b));
    }
    return pack_bf16x2(ya, yb);
}

template <int kAct>
__device__ __forceinline__ void frag_stage(const uint32_t (&lo)[8], const uint32_t (&hi)[8], uint32_t row_addr) {
    stmatrix_x4_trans(row_addr, frag_pack<kAct>(lo[0], lo[1]), frag_pack<kAct>(lo[2], lo[3]), frag_pack<kAct>(lo[4], lo[5]),
                      frag_pack<kAct>(lo[6], lo[7]));
    stmatrix_x4_trans(row_addr + 32u, frag_pack<kAct>(hi[0], hi[1]), frag_pack<kAct>(hi[2], hi[3]), frag_pack<kAct>(hi[4], hi[5]),
                      frag_pack<kAct>(hi[6], hi[7]));
}

// taddr: this warp's lane quadrant, first column of the accumulator.  16 token columns per step; the loads of the next
// step are in flight while the current one is converted and stored.
__device__ __forceinline__ void drain_direct_frag(uint32_t taddr, int total, uint32_t bar_release, const EmitCtx& e, uint32_t& parity) {
    const int begin = 0;
    const int lane = e.r & 31, wq = e.r >> 5;
    // stmatrix row address of this thread: matrix i = lane / 8 covers tokens 8 (i / 2) .. + 7 and features 8 (i % 2) .. + 7 of
    // the 16-lane half; row j = lane % 8 is token 8 (i / 2) + j
    const uint32_t row_off = static_cast<uint32_t>(((lane >> 4) * 8 + (lane & 7)) * kFragPitch + (wq * 32 + ((lane >> 3) & 1) * 8) * 2);
    uint32_t la[8], ha[8], lb[8], hb[8];
    tmem_ld_16x256b_x2(taddr + begin, la);
    tmem_ld_16x256b_x2(taddr + (16u << 16) + begin, ha);
    for (int cc = begin; cc < total; cc += 32) {
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            const int c0 = cc + 16 * half;
            if (c0 >= total) break;
            tmem_ld_wait();
            const bool more = c0 + 16 < total;
            uint32_t (&lo)[8] = half == 0 ? la : lb;
            uint32_t (&hi)[8] = half == 0 ? ha : hb;
            uint32_t (&nlo)[8] = half == 0 ? lb : la;
            uint32_t (&nhi)[8] = half == 0 ? hb : ha;
            if (more) {
                tmem_ld_16x256b_x2(taddr + c0 + 16, nlo);
                tmem_ld_16x256b_x2(taddr + (16u << 16) + c0 + 16, nhi);
            } else {
                release_acc(bar_release);
            }
            const uint32_t buf = e.stage_s + (parity & 1u) * kStageBufBytes;
            parity ^= 1u;
            if (e.act == kActGeluTanh) frag_stage<kActGeluTanh>(lo, hi, buf + row_off);
            else if (e.act == kActRelu) frag_stage<kActRelu>(lo, hi, buf + row_off);
            else frag_stage<kActNone>(lo, hi, buf + row_off);
            bar_sync(1, kEpiThreads);
            const int rr = c0 >= e.tile_m ? 1 : 0, c = c0 - rr * e.tile_m;
            const int n_base = e.n_first + rr * kTileN, m_first = e.m0 + c;
            uint4 v[2];
#pragma unroll
            for (int p = 0; p < 2; ++p) {
                const int piece = p * kEpiThreads + e.r;  // 16 pieces of 8 features per token row
                v[p] = ld_shared_v4(buf + static_cast<uint32_t>(piece >> 4) * kFragPitch + static_cast<uint32_t>(piece & 15) * 16u);
            }
#pragma unroll
            for (int p = 0; p < 2; ++p) {
                const int piece = p * kEpiThreads + e.r;
                const int m = m_first + (piece >> 4), n = n_base + (piece & 15) * 8;
                if (m < e.m_end && n < e.N) *reinterpret_cast<uint4*>(e.out + static_cast<size_t>(m) * e.ld + n) = v[p];
            }
        }
    }
}

// Drain one accumulator (`total` TMEM columns from taddr) in chunks of kC columns: the tcgen05.ld of the next
// chunk is in flight while the current one is consumed -- kDirect: act + bf16 + transposed store of the output
// (steps a3 / a7), else: fp32 split-K partial (step a8); once the last chunk has been read the accumulator is
// handed back to the MMA warp (bar_release = tempty).
template <int kC, bool kDirect>
__device__ __forceinline__ void drain_acc(uint32_t taddr, int total, uint32_t bar_release, const EmitCtx& e, uint32_t& parity,
                                          float* wsp) {
    uint32_t va[kC], vb[kC];
    tmem_ld_cols<kC>(taddr, va);
    for (int cc = 0; cc < total; cc += 2 * kC) {
        tmem_ld_wait();
        const bool more = cc + kC < total;
        if (more) tmem_ld_cols<kC>(taddr + cc + kC, vb);
        else release_acc(bar_release);
        if (kDirect) emit_chunk<kC>(va, cc, e, parity);
        else store_chunk<kC>(va, cc, wsp);
        if (more) {
            tmem_ld_wait();
            if (cc + 2 * kC < total) tmem_ld_cols<kC>(taddr + cc + 2 * kC, va);
            else release_acc(bar_release);
            if (kDirect) emit_chunk<kC>(vb, cc + kC, e, parity);
            else store_chunk<kC>(vb, cc + kC, wsp);
        }
    }
}

__device__ __forceinline__ void st_relaxed_gpu(uint32_t* p, uint32_t v) {
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Table entry of ticket t as the two words of a UnitDesc; computed when the layer's first tickets follow the
// closed form (static_sp), else read.
__device__ __forceinline__ uint2 unit_words(const LayerParams& L, uint32_t t, bool may_compute) {
    if (may_compute && L.static_sp > 0) {
        const uint32_t sp = static_cast<uint32_t>(L.static_sp), tile = t / sp, ks = t % sp;
        const uint32_t a = ks * static_cast<uint32_t>(L.kb_total) / sp, b = (ks + 1) * static_cast<uint32_t>(L.kb_total) / sp;
        return make_uint2(tile | (static_cast<uint32_t>(kUnitMma) << 16) | (ks << 24), a | (b << 16));
    }
    return __ldg(reinterpret_cast<const uint2*>(L.table) + t);
}

// Watchdog expiry: record it in the device status word (every other waiter then gives up after its next 256 polls) and in
// the pinned host mirror, where the next mlp_pipe_run on the handle finds it without a device round trip.
__device__ __forceinline__ void flag_timeout(uint32_t* status, uint32_t* status_host) {
    if (atomicCAS(status, 0u, kStatusFlagTimeout) == 0u && status_host) {
        *reinterpret_cast<volatile uint32_t*>(status_host) = kStatusFlagTimeout;
        __threadfence_system();
    }
}

// Spin until *ctr has reached `target` (wrap-safe), then acquire.  Relaxed polls + one acquire fence =
// acquire pattern.  Bounded: after timeout_ns (or when another waiter has already given up) the wait is
// abandoned, the device status word records it and the caller carries on (output undefined, kernel ends).
__device__ __forceinline__ void poll_counter(const uint32_t* ctr, uint32_t target, uint32_t* status, uint32_t* status_host,
                                             unsigned long long timeout_ns, unsigned long long& waited) {
    if (static_cast<int32_t>(ld_relaxed_gpu(ctr) - target) < 0) {
        const long long c0 = clock64();
        const uint64_t t0 = globaltimer_ns();
        uint32_t n = 0;
        while (static_cast<int32_t>(ld_relaxed_gpu(ctr) - target) < 0) {
            __nanosleep(32);
            if ((++n & 255u) == 0) {
                if (ld_relaxed_gpu(status) != 0) break;
                if (globaltimer_ns() - t0 > timeout_ns) {
                    flag_timeout(status, status_host);
                    break;
                }
            }
        }
        waited += static_cast<unsigned long long>(clock64() - c0);
    }
    fence_acq_rel_gpu();
}

// arrive on the barrier at this offset in the pair LEADER's shared memory (own barrier when not in pair mode)
__device__ __forceinline__ void arrive_leader(uint32_t bar, bool pair) {
    if (pair) mbar_arrive_cluster(bar & kPeerBitMask);
    else mbar_arrive(bar);
}
// wait on an own barrier that the other CTA of the pair may arrive on (acquire at cluster scope then)
__device__ __forceinline__ void wait_shared(uint32_t bar, uint32_t parity, bool pair) {
    if (pair) mbar_wait_cluster(bar, parity);
    else mbar_wait(bar, parity);
}

// kPair: the CTA-pair build (tcgen05 cta_group::2).  A separate instantiation because a kernel that contains cta_group::2
// instructions can only be launched in clusters of two.
template <bool kPair>
__global__ void __launch_bounds__(kThreads, 1) mlp_pipe_kernel(const __grid_constant__ KernelParams P) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));

    const int tile_m = P.tile_m;
    constexpr bool pair = kPair;
    const uint32_t rank = pair ? cluster_ctarank() : 0u;   // rank in the CTA pair; the leader is rank 0
    const bool leader = rank == 0;
    const int nb_mul = pair ? 2 : 1;                       // 128-row counter tiles per table tile
    const int a_rows = pair ? tile_m / 2 : tile_m;         // token rows of the activation tile this CTA stages
    const int n_sub = P.n_sub;
    const int tile_n = kTileN * n_sub;  // weight rows per unit
    const uint32_t w_tile_bytes = static_cast<uint32_t>(n_sub) * kWTileBytes;
    const uint32_t a_tile_bytes = static_cast<uint32_t>(a_rows) * (kTileK * 2);
    const int stages = P.stages;      // weight ring depth
    const int a_stages = P.a_stages;  // activation ring depth (= stages unless mlp_mode.a_stages asks otherwise)
    // Equally deep rings share their barriers: "stage s landed" counts the bytes of both tiles (two arrivals, one per
    // loader), "stage s consumed" is ONE commit that both loaders wait for -- one wait and one commit per K-block.
    const bool unified = stages == a_stages;
    const uint32_t a_ring = smem_base + static_cast<uint32_t>(stages) * w_tile_bytes;
    const uint32_t stage_s = a_ring + static_cast<uint32_t>(a_stages) * a_tile_bytes;  // epilogue staging
    const uint32_t ring_bytes = static_cast<uint32_t>(stages) * w_tile_bytes + static_cast<uint32_t>(a_stages) * a_tile_bytes + kStageBytes;

    // control block after the rings
    uint8_t* ctrl = smem_gen + ring_bytes;
    const uint32_t ctrl_s = smem_base + ring_bytes;
    const uint32_t bar_full = ctrl_s;                          // [kMaxStages]  weight tile landed
    const uint32_t bar_empty = bar_full + 8 * kMaxStages;      // [kMaxStages]  weight stage consumed
    const uint32_t bar_afull = unified ? bar_full : bar_empty + 8 * kMaxStages;     // [kMaxStages]  activation tile landed
    const uint32_t bar_aempty = unified ? bar_empty : bar_empty + 16 * kMaxStages;  // [kMaxStages]  activation stage consumed
    const uint32_t bar_tfull = bar_full + 32 * kMaxStages;     // [kMaxAccStages]
    const uint32_t bar_tempty = bar_tfull + 8 * kMaxAccStages;  // [kMaxAccStages]
    const uint32_t bar_sfull = bar_tempty + 8 * kMaxAccStages;  // [kSchedSlots]
    const uint32_t bar_sempty = bar_sfull + 8 * kSchedSlots;   // [kSchedSlots]
    const uint32_t bar_wtaken = bar_sempty + 8 * kSchedSlots;  // [kSchedSlots]
    constexpr int kBarBytes = 8 * (4 * kMaxStages + 2 * kMaxAccStages + 3 * kSchedSlots);
    UnitInfo* ring = reinterpret_cast<UnitInfo*>(ctrl + kBarBytes);
    volatile uint32_t* s_tmem = reinterpret_cast<volatile uint32_t*>(ctrl + kBarBytes + sizeof(UnitInfo) * kSchedSlots);
    volatile uint32_t* s_last = s_tmem + 1;
    volatile unsigned long long* s_epoch = reinterpret_cast<volatile unsigned long long*>(s_tmem + 2);
    volatile uint32_t* s_pre = s_tmem + 4;  // [0] weight / [1] activation K-blocks of the first unit requested during setup,
                                            // [2] 1 if the first unit already sits in slot 0 of the scheduler ring

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const long long t_start = clock64();
    CtaStats* const my_stats = P.stats + blockIdx.x;
    if (threadIdx.x == 0) my_stats->ts[0] = globaltimer_ns();

    // TMEM accumulator ring: as many (n_sub x tile_m)-column accumulators as fit (<= 8), so that the MMA
    // warp can run ahead of an epilogue that is waiting on a memory round trip
    const uint32_t acc_stages = static_cast<uint32_t>(P.acc_stages);
    const uint32_t acc_cols = static_cast<uint32_t>(n_sub * tile_m);
    uint32_t tmem_cols = 32;
    while (tmem_cols < acc_stages * acc_cols) tmem_cols <<= 1;

    // ------------------------------------------------------------------ one-time setup
    if (threadIdx.x == 0) {
        if (P.flags & kFlagPdl) grid_launch_dependents();
        // device-resident epoch: no per-run host state, so a captured graph can be replayed
        *s_epoch = ld_relaxed_gpu_u64(reinterpret_cast<const uint64_t*>(P.epoch_counter)) / gridDim.x;
        for (int l = P.layer_begin; l < P.layer_end; ++l) {
            prefetch_tmap(&P.tm_w[l]);
            prefetch_tmap(&P.tm_a[l]);
        }
    }
    if (warp == 1) {
        // All mbarriers live in one array of 8-byte slots; the 32 lanes of the weight-loader warp initialise them in
        // parallel (92 serial mbarrier.init cost ~1 us at the head of every CTA), arrival counts by slot range.
        constexpr int kNumBars = 4 * kMaxStages + 2 * kMaxAccStages + 3 * kSchedSlots;
        for (int b = lane; b < kNumBars; b += 32) {
            uint32_t count = (unified && b < kMaxStages) ? 2u : 1u;                                                                   // full (unified: W loader + A loader)
            if (b >= 4 * kMaxStages + kMaxAccStages && b < 4 * kMaxStages + 2 * kMaxAccStages) count = kEpiThreads * nb_mul;          // tempty (pair: both CTAs' epilogues)
            if (b >= 4 * kMaxStages + 2 * kMaxAccStages + kSchedSlots && b < 4 * kMaxStages + 2 * kMaxAccStages + 2 * kSchedSlots)
                count = (3 + kEpiThreads) * nb_mul;                                                                                   // sempty (pair: both CTAs' consumers)
            mbar_init(bar_full + 8 * b, count);
        }
        fence_mbar_init();
        fence_proxy_async();  // the inits (generic proxy) before the TMA unit's complete_tx on them
        __syncwarp();
    }
    if (threadIdx.x == 32) {
        // This thread is the weight loader.  The first unit of the CTA is static (same rule as in the
        // scheduler below), so its first ring of weight tiles -- and, if it has no producers, of activation
        // tiles -- is requested right here, before TMEM allocation and the CTA-wide sync: the first bytes are
        // in flight ~1 us earlier.
        int l0 = P.layer_begin;
        uint32_t sid = blockIdx.x;
        if (static_cast<int>(blockIdx.x) >= P.producer_ctas && P.layer_begin + 1 < P.layer_end) {
            l0 = P.layer_begin + 1;
            sid = blockIdx.x - P.producer_ctas;
        }
        const bool have = !pair && sid < static_cast<uint32_t>(P.layer[l0].units) &&
                          !(P.layer[l0].use_queue && P.wait_flags && l0 > P.layer_begin);  // (a queue-mode unit is unknown until popped)
        uint2 raw = make_uint2(0u, 0u);
        prefetch_tmap(&P.tm_w[l0]);
        prefetch_tmap(&P.tm_a[l0]);
        if (have) raw = unit_words(P.layer[l0], sid, true);
        fence_mbar_init();
        uint32_t pre_w = 0, pre_a = 0;
        if (have && ((raw.x >> 16) & 0xffu) == kUnitMma && !(P.flags & kFlagExpNoPreissue)) {
            fence_proxy_async();  // the barrier inits (generic proxy) before the TMA unit's complete_tx on them
            const int tile = static_cast<int>(raw.x & 0xffffu), kb0 = static_cast<int>(raw.y & 0xffffu), kb1 = static_cast<int>(raw.y >> 16);
            const int n_blk = tile % P.layer[l0].n_blks, m_blk = tile / P.layer[l0].n_blks;
            const uint64_t pol = policy_evict_first();
            pre_w = static_cast<uint32_t>(min(stages, kb1 - kb0));
            my_stats->ts[3] = globaltimer_ns();
            for (uint32_t i = 0; i < pre_w; ++i) {
                mbar_arrive_expect_tx(bar_full + 8 * i, w_tile_bytes);
                if (!(P.flags & kFlagNoEvictFirst))
                    tma_load_2d_hint(smem_base + i * w_tile_bytes, &P.tm_w[l0], (kb0 + static_cast<int>(i)) * kTileK, n_blk * tile_n, bar_full + 8 * i, pol);
                else tma_load_2d(smem_base + i * w_tile_bytes, &P.tm_w[l0], (kb0 + static_cast<int>(i)) * kTileK, n_blk * tile_n, bar_full + 8 * i);
            }
            if (l0 == P.layer_begin && !P.pdl_wait && !P.wait_first) {  // input of the launch: nothing to wait for
                pre_a = static_cast<uint32_t>(min(min(a_stages, stages), kb1 - kb0));
                for (uint32_t i = 0; i < pre_a; ++i) {
                    mbar_arrive_expect_tx(bar_afull + 8 * i, a_tile_bytes);
                    tma_load_2d(a_ring + i * a_tile_bytes, &P.tm_a[l0], (kb0 + static_cast<int>(i)) * kTileK, P.m_off + m_blk * tile_m, bar_afull + 8 * i);
                }
            }
        }
        s_pre[0] = pre_w;
        s_pre[1] = pre_a;
        // ... and the unit itself goes into slot 0 of the scheduler ring right away, so that after the CTA-wide sync
        // the MMA / loader / epilogue warps start on it without waiting for the scheduler warp
        s_pre[2] = have ? 1u : 0u;
        if (have) {
            UnitInfo u;
            u.layer = l0;
            u.tile = static_cast<int>(raw.x & 0xffffu);
            u.kind = static_cast<int>((raw.x >> 16) & 0xffu);
            u.ks = static_cast<int>(raw.x >> 24);
            u.kb0 = static_cast<int>(raw.y & 0xffffu);
            u.kb1 = static_cast<int>(raw.y >> 16);
            u.m_blk = u.tile / P.layer[l0].n_blks;
            u.n_blk = u.tile % P.layer[l0].n_blks;
            u.valid = 1;
            u.acquired = 0;  // a consumer-first or reduce unit polls for itself
            u.pad_[0] = u.pad_[1] = 0;
            ring[0] = u;
            mbar_arrive(bar_sfull);  // slot 0 (release: the slot is visible to the waiters)
        }
    }
    if (warp == 3) {
        if (pair) {  // the same warp of both CTAs allocates the same columns in both TMEMs
            tmem_alloc_pair(smem_u32(const_cast<uint32_t*>(s_tmem)), tmem_cols);
            tmem_relinquish_pair();
        } else {
            tmem_alloc(smem_u32(const_cast<uint32_t*>(s_tmem)), tmem_cols);
            tmem_relinquish();
        }
    }
    tc_fence_before();
    if (pair) cluster_sync_all();  // the peer's barriers are initialised before anything arrives on them remotely
    else __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *s_tmem;
    const unsigned long long epoch = *s_epoch;
    if (threadIdx.x == 0) my_stats->ts[1] = globaltimer_ns();

    // ------------------------------------------------------------------ roles
    if (warp == 0) {
        // ===== scheduler: ticket -> unit (step a1, ordering knob PAPER.md:99-101); in pair mode only
        // the leader CTA schedules and hands every unit to both CTAs' rings
        if (lane == 0 && leader) {
            uint32_t done[kMaxLayers];
            for (int l = 0; l < kMaxLayers; ++l) done[l] = 0;
            unsigned long long q_stall = 0, q_polls = 0;
            int l = P.layer_begin;
            // the first unit of a CTA is static (its rank among the CTAs that start on the same layer):
            // no atomic round trip before the first weight load
            uint32_t static_id = blockIdx.x / nb_mul;  // worker index (a worker = a CTA, or a CTA pair)
            bool use_static = true;
            if (static_cast<int>(static_id) >= P.producer_ctas && P.layer_begin + 1 < P.layer_end) {
                l = P.layer_begin + 1;
                static_id -= P.producer_ctas;
            }
            uint32_t it = 0;
            bool finished = false;
            if (s_pre[2]) {  // the static first unit was published by the weight loader during setup
                use_static = false;
                done[l] = 1;
                it = 1;
                my_stats->ts[2] = globaltimer_ns();
            }
            while (!finished) {
                UnitInfo u;
                u.valid = 0;
                u.layer = u.m_blk = u.n_blk = u.ks = u.kb0 = u.kb1 = u.tile = u.acquired = u.kind = 0;
                // claim at most one unit ahead of the W loader (keeps the tail balanced)
                if (it >= 1) mbar_wait(bar_wtaken + 8 * ((it - 1) % kSchedSlots), ((it - 1) / kSchedSlots) & 1);
                while (l < P.layer_end) {
                    const LayerParams& L = P.layer[l];
                    uint32_t t;
                    const bool is_static = use_static;  // only the static ticket lies in the prefix the host verified against the closed form
                    if (use_static) {
                        use_static = false;
                        t = static_id;
                    } else {
                        const uint32_t base = static_cast<uint32_t>(epoch * static_cast<unsigned long long>(L.ticket_inc));
                        t = atom_add_relaxed_gpu(L.ticket, 1u) - base + static_cast<uint32_t>(L.ticket_off);
                    }
                    if (t >= static_cast<uint32_t>(L.units)) {
                        ++l;
                        continue;
                    }
                    uint2 raw;
                    bool popped = false;
                    if (L.use_queue && P.wait_flags && l > P.layer_begin) {
                        // Consumer prologue of the paper's protocol (PAPER.md:95 step (5)): ticket t is a
                        // POSITION in the work queue; spin until a producer has pushed an entry there, then remap
                        // the unit ("tile id") to what the entry names.  Entries appear in the order in which groups
                        // of units became ready, so the unit -- and with it the weights to prefetch -- is not known
                        // before the pop.
                        const uint32_t tag = static_cast<uint32_t>(epoch + 1ull) & 0xffffu;
                        uint32_t v = ld_relaxed_gpu(L.queue + t);
                        if ((v >> 16) != tag) {
                            const long long c0 = clock64();
                            const uint64_t t0 = globaltimer_ns();
                            uint32_t n = 0;
                            bool gave_up = false;
                            while (((v = ld_relaxed_gpu(L.queue + t)) >> 16) != tag) {
                                __nanosleep(32);
                                if ((++n & 255u) == 0) {
                                    if (ld_relaxed_gpu(P.status) != 0) { gave_up = true; break; }
                                    if (globaltimer_ns() - t0 > P.timeout_ns) {
                                        flag_timeout(P.status, P.status_host);
                                        gave_up = true;
                                        break;
                                    }
                                }
                            }
                            q_stall += static_cast<unsigned long long>(clock64() - c0);
                            q_polls += n;
                            if (gave_up) v = t;  // watchdog: fall back to the static order so that the kernel terminates
                        }
                        fence_acq_rel_gpu();  // acquire: the pusher released after the last producer tile of the group
                        raw = __ldg(reinterpret_cast<const uint2*>(L.table) + (v & 0xffffu));
                        popped = true;
                    } else {
                        raw = unit_words(L, t, is_static);
                    }
                    u.layer = l;
                    u.tile = static_cast<int>(raw.x & 0xffffu);
                    u.kind = static_cast<int>((raw.x >> 16) & 0xffu);
                    u.ks = static_cast<int>(raw.x >> 24);
                    u.kb0 = static_cast<int>(raw.y & 0xffffu);
                    u.kb1 = static_cast<int>(raw.y >> 16);
                    u.m_blk = u.tile / L.n_blks;
                    u.n_blk = u.tile % L.n_blks;
                    u.valid = 1;
                    if (popped) {
                        u.acquired = 1;
                    } else if (u.kind == kUnitReduce && pair) {
                        // each CTA of the pair reduces its own 128 rows and polls its own arrival counter
                    } else if (u.kind == kUnitReduce) {
                        // fast path of a reduce unit: all slices of its tile have already arrived
                        const uint32_t target = static_cast<uint32_t>((epoch + 1ull) * static_cast<unsigned long long>(L.split));
                        if (static_cast<int32_t>(ld_relaxed_gpu(L.arrive + u.tile) - target) >= 0) {
                            fence_acq_rel_gpu();
                            u.acquired = 1;
                        }
                    } else if (P.wait_flags && (l > P.layer_begin || P.wait_first) && !(P.flags & (kFlagExpNoFastPath | kFlagAcquireLoads))) {
                        // Consumer prologue, fast path (the prologue lives in the scheduler
                        // warp): one look at all ready counters under this unit's K range.  If every producer
                        // tile is already published -- the normal case, the scheduler runs a unit ahead --
                        // ONE acquire fence here covers the whole unit and the loaders never poll.  Otherwise
                        // the activation loader polls slice by slice while the weight loader prefetches.
                        const LayerParams& Lp = P.layer[l - 1];
                        const uint32_t target = static_cast<uint32_t>((epoch + 1ull) * static_cast<unsigned long long>(Lp.ready_inc));
                        // (pair mode: the counters are per 128-row block, tile_n = 128 here, and the acquire reaches the peer's
                        // loaders through the cluster-scope release / acquire of the slot hand-over: causality order is transitive)
                        const uint32_t* rd = Lp.ready + u.m_blk * Lp.n_blks * nb_mul;
                        const int s0 = (u.kb0 * kTileK) / tile_n, s1 = ((u.kb1 - 1) * kTileK) / tile_n + 1;
                        bool all = (s1 - s0) <= 256;  // (the scheduler runs a unit ahead: its round trips are off the critical path)
                        for (int sb = s0; sb < s1 && all; sb += 8) {
                            uint32_t v[8];
#pragma unroll
                            for (int i = 0; i < 8; ++i) v[i] = (sb + i < s1) ? ld_relaxed_gpu(rd + sb + i) : target;
#pragma unroll
                            for (int i = 0; i < 8; ++i) all = all && static_cast<int32_t>(v[i] - target) >= 0;
                        }
                        if (all) {
                            fence_acq_rel_gpu();
                            u.acquired = 1;
                        }
                    }
                    if (it == 0) my_stats->ts[2] = globaltimer_ns();
                    done[l]++;
                    break;
                }
                finished = !u.valid;
                const uint32_t slot = it % kSchedSlots;
                if (it >= kSchedSlots) wait_shared(bar_sempty + 8 * slot, ((it / kSchedSlots) & 1) ^ 1, pair);
                ring[slot] = u;
                if (pair) {  // the same slot of the peer's ring, then both "slot full" barriers (release at cluster scope)
                    const uint32_t peer_slot = mapa_u32(smem_u32(&ring[slot]), 1u);
                    const uint32_t* w = reinterpret_cast<const uint32_t*>(&u);
#pragma unroll
                    for (int i = 0; i < static_cast<int>(sizeof(UnitInfo) / 4); ++i) st_cluster_u32(peer_slot + 4 * i, w[i]);
                    mbar_arrive_cluster(mapa_u32(bar_sfull + 8 * slot, 1u));
                    mbar_arrive_cluster(bar_sfull + 8 * slot);
                } else {
                    mbar_arrive(bar_sfull + 8 * slot);  // release: ring[slot] visible to waiters
                }
                ++it;
            }
            for (int l2 = 0; l2 < kMaxLayers; ++l2) P.stats[blockIdx.x].units[l2] = done[l2];
            if (P.flags & kFlagWorkQueue) {  // (the activation loader never polls in this mode)
                my_stats->stall_cycles = q_stall;
                my_stats->polls = q_polls;
            }
        }
    } else if (warp == 1) {
        // ===== W loader: all 32 lanes run the loop converged and wait, one elected lane issues.  (Measured: what makes a
        // converged role slow is divergence INSIDE its loop -- a probe-then-wait branch per stage, `if (lane == 0)` arrivals,
        // or worst of all one lane waiting while the others sit at a __syncwarp (cfg 1 66 instead of 51 us); with plain waits
        // and every single-lane action under elect.sync it beats the one-thread form: cfg 1 mean 50.7 vs 51.4 us.)
        {
            const uint64_t pol = policy_evict_first();
            const bool hint = !(P.flags & kFlagNoEvictFirst);
            uint32_t stage = 0, phase = 0;
            unsigned long long w_wait = 0;  // cycles inside the waits for a free stage (a wait that succeeds at once costs ~100)
            for (uint32_t it = 0;; ++it) {
                const uint32_t slot = it % kSchedSlots;
                wait_shared(bar_sfull + 8 * slot, (it / kSchedSlots) & 1, pair);
                const UnitInfo u = ring[slot];
                __syncwarp();  // every lane holds the unit before the slot is handed back
                // Late binding: the scheduler may draw the NEXT ticket only once this unit has at most
                // claim_ahead K-blocks left to request.  A unit stalled on its producers (the ring is full, the
                // MMA warp waits for the activation loader) therefore never holds a second ticket.
                // (For a reduce unit the epilogue warps give the go once its partials have arrived.)
                bool told = u.kind == kUnitReduce || !u.valid || u.kb1 - u.kb0 <= P.claim_ahead;
                if (elect_one()) {
                    arrive_leader(bar_sempty + 8 * slot, pair);
                    if (told && u.kind != kUnitReduce) mbar_arrive(bar_wtaken + 8 * slot);
                    if (u.valid && it < kUnitTrace) {
                        const uint64_t now = globaltimer_ns();
                        my_stats->unit_ts[it][0] = now;
                        if (u.kind == kUnitReduce) my_stats->unit_ts[it][1] = now;
                        my_stats->unit_id[it] = (static_cast<uint32_t>(u.layer) << 28) | (static_cast<uint32_t>(u.tile) << 8) |
                                                static_cast<uint32_t>(u.kind == kUnitReduce ? 0x80 | (u.kb0 >> 4) : u.ks);
                    }
                }
                __syncwarp();
                if (!u.valid) break;
                if (u.kind == kUnitReduce) continue;
                const CUtensorMap* tm = &P.tm_w[u.layer];
                // K-blocks are requested in groups of w_group: the loader first waits until the whole group of
                // stages is free and then issues the group back to back, so that the 128-byte pieces of one
                // weight row that are adjacent in memory reach the DRAM controller together
                int kb = u.kb0;
                if (it == 0) {  // the first ring of this unit was requested during setup
                    const uint32_t pre = s_pre[0];
                    kb += static_cast<int>(pre);
                    stage = pre % static_cast<uint32_t>(stages);
                    phase = pre / static_cast<uint32_t>(stages);
                }
                const int w_row = pair ? (u.n_blk * 2 + static_cast<int>(rank)) * kTileN : u.n_blk * tile_n;
                while (kb < u.kb1) {
                    const int g = min(P.w_group, u.kb1 - kb);
                    uint32_t st = stage, ph = phase;
                    const long long t0 = clock64();
                    for (int i = 0; i < g; ++i) {
                        mbar_wait(bar_empty + 8 * st, ph ^ 1);
                        if (++st == static_cast<uint32_t>(stages)) { st = 0; ph ^= 1; }
                    }
                    w_wait += static_cast<unsigned long long>(clock64() - t0);
                    const bool tell = !told && u.kb1 - kb <= P.claim_ahead;
                    told = told || tell;
                    for (int i = 0; i < g; ++i, ++kb) {
                        const uint32_t full = bar_full + 8 * stage;
                        const uint32_t dst = smem_base + stage * w_tile_bytes;
                        if (elect_one()) {
                            if (tell && i == 0) mbar_arrive(bar_wtaken + 8 * slot);
                            if (pair) {
                                // each CTA loads its own 128 weight rows; the bytes of BOTH count on the leader's barrier
                                if (leader) mbar_arrive_expect_tx(full, 2 * w_tile_bytes);
                                tma_load_2d_pair(dst, tm, kb * kTileK, w_row, full, pol);
                            } else {
                                mbar_arrive_expect_tx(full, w_tile_bytes);
                                if (hint) tma_load_2d_hint(dst, tm, kb * kTileK, w_row, full, pol);
                                else tma_load_2d(dst, tm, kb * kTileK, w_row, full);
                            }
                        }
                        __syncwarp();
                        if (++stage == static_cast<uint32_t>(stages)) { stage = 0; phase ^= 1; }
                    }
                }
                if (it < kUnitTrace && elect_one()) my_stats->unit_ts[it][1] = globaltimer_ns();
                __syncwarp();
            }
            if (lane == 0) my_stats->wait[0] = w_wait;
        }
    } else if (warp == 2) {
        // ===== A loader = consumer prologue (step a5; PAPER.md:95 step (5))
        // (all lanes converged: every lane polls, fences and waits; one elected lane issues the TMA)
        {
            uint32_t stage = 0, phase = 0;
            unsigned long long stall = 0, polls = 0;
            bool aborted = false;
            const uint64_t pol_a = policy_evict_normal();
            if (P.pdl_wait) {
                // programmatic dependent launch (stronger SEQUENTIAL baseline): this grid was allowed to start while
                // the grid of the layer before still runs; setup and the weight prefetch overlap its tail, and only
                // here -- before the first read of what it wrote -- do we wait for its completion
                grid_dependency_wait();
                fence_proxy_async();
            }
            for (uint32_t it = 0;; ++it) {
                const uint32_t slot = it % kSchedSlots;
                wait_shared(bar_sfull + 8 * slot, (it / kSchedSlots) & 1, pair);
                const UnitInfo u = ring[slot];
                __syncwarp();  // every lane holds the unit before the slot is handed back
                if (lane == 0) arrive_leader(bar_sempty + 8 * slot, pair);
                if (!u.valid) break;
                if (u.kind == kUnitReduce) continue;
                const CUtensorMap* tm = &P.tm_a[u.layer];
                const int a_row = P.m_off + u.m_blk * tile_m + (pair ? static_cast<int>(rank) * a_rows : 0);
                const bool consumer = P.wait_flags && (u.layer > P.layer_begin || P.wait_first);
                const bool wait = consumer && !u.acquired;
                if (consumer) fence_proxy_async();
                const LayerParams& Lp = P.layer[u.layer > 0 ? u.layer - 1 : 0];
                const uint32_t target = static_cast<uint32_t>((epoch + 1ull) * static_cast<unsigned long long>(Lp.ready_inc));
                const uint32_t* ready = wait ? Lp.ready + u.m_blk * Lp.n_blks * nb_mul : nullptr;
                // Slices [.., ready_upto) of this unit are known to be published.  Readiness is monotone
                // within a run, so the prologue looks ahead: up to 8 counters are read with independent
                // relaxed loads that are ISSUED a few K-blocks before their result is needed (the round trip
                // overlaps the TMA issue of slices already known to be ready), then one acquire fence turns
                // the observations into an acquire pattern (PTX memory model: relaxed read + fence.acq_rel).
                const int slice_end = wait ? ((u.kb1 - 1) * kTileK) / tile_n + 1 : 0;
                int ready_upto = wait ? (u.kb0 * kTileK) / tile_n : 0;
                uint32_t v[8];
                int pend_base = -1;  // >= 0: v[] holds in-flight reads of counters pend_base .. pend_base+7
                int kb_first = u.kb0;
                if (it == 0) {
                    const uint32_t pre = s_pre[1];
                    kb_first += static_cast<int>(pre);
                    stage = pre % static_cast<uint32_t>(a_stages);
                    phase = pre / static_cast<uint32_t>(a_stages);
                }
                for (int kb = kb_first; kb < u.kb1; ++kb) {
                    mbar_wait(bar_aempty + 8 * stage, phase ^ 1);
                    if (wait) {
                        const int slice = (kb * kTileK) / tile_n;  // producer tile that wrote these columns
                        if (pend_base < 0 && ready_upto < slice_end && slice + 2 >= ready_upto) {
                            pend_base = ready_upto;
#pragma unroll
                            for (int i = 0; i < 8; ++i)
                                v[i] = (pend_base + i < slice_end) ? ((P.flags & kFlagAcquireLoads) ? ld_acquire_gpu(ready + pend_base + i) : ld_relaxed_gpu(ready + pend_base + i)) : target - 1u;
                        }
                        if (slice >= ready_upto) {
                            int n_ok = 0;
#pragma unroll
                            for (int i = 0; i < 8; ++i)
                                if (n_ok == i && static_cast<int32_t>(v[i] - target) >= 0) n_ok = i + 1;
                            if (n_ok == 0) {
                                if (!aborted) {
                                    const long long c0 = clock64();
                                    const uint64_t t0 = globaltimer_ns();
                                    uint32_t n = 0;
                                    while (static_cast<int32_t>(((P.flags & kFlagAcquireLoads) ? ld_acquire_gpu(ready + slice) : ld_relaxed_gpu(ready + slice)) - target) < 0) {
                                        ++n;
                                        __nanosleep(32);
                                        if ((n & 255u) == 0) {
                                            if (ld_relaxed_gpu(P.status) != 0) { aborted = true; break; }
                                            if (globaltimer_ns() - t0 > P.timeout_ns) {
                                                if (lane == 0) flag_timeout(P.status, P.status_host);
                                                aborted = true;
                                                break;
                                            }
                                        }
                                    }
                                    polls += n;
                                    stall += static_cast<unsigned long long>(clock64() - c0);
                                }
                                n_ok = 1;
                            }
                            if (!(P.flags & (kFlagExpNoAcquireFence | kFlagAcquireLoads))) fence_acq_rel_gpu();
                            // H was written through the generic proxy; the TMA below reads it through
                            // the async proxy
                            if (!(P.flags & kFlagExpNoProxyFence)) fence_proxy_async();
                            ready_upto = pend_base + n_ok;
                            pend_base = -1;
                        }
                    }
                    if (elect_one()) {
                        if (pair) {  // each CTA stages HALF of the tokens (the B operand of the pair MMA is split between the CTAs)
                            if (leader) mbar_arrive_expect_tx(bar_afull + 8 * stage, 2 * a_tile_bytes);
                            tma_load_2d_pair(a_ring + stage * a_tile_bytes, tm, kb * kTileK, a_row, bar_afull + 8 * stage, pol_a);
                        } else {
                            mbar_arrive_expect_tx(bar_afull + 8 * stage, a_tile_bytes);
                            tma_load_2d(a_ring + stage * a_tile_bytes, tm, kb * kTileK, a_row, bar_afull + 8 * stage);
                        }
                    }
                    __syncwarp();
                    if (++stage == static_cast<uint32_t>(a_stages)) { stage = 0; phase ^= 1; }
                }
            }
            if (!(P.flags & kFlagWorkQueue) && lane == 0) {
                P.stats[blockIdx.x].stall_cycles = stall;
                P.stats[blockIdx.x].polls = polls;
            }
        }
    } else if (warp == 3) {
        // ===== MMA issuer (steps a2, a6).  All 32 lanes run the loop CONVERGED and wait on the barriers; one elected lane
        // issues.  (A lone `lane == 0` thread makes ptxas wrap every tcgen05 instruction into an elect / branch loop over
        // the active lanes, and the round trip of each mbarrier test then sits between two MMAs: measured 858 cycles per
        // K-block of 4 MMAs + 2 waits + 2 commits against a tensor-core floor of 512 at N = 256 -- the pipe was paced by
        // its issuer.  Converged, with ONE wait and ONE commit per K-block where the rings are equally deep: 424.)
        {
            // pair mode: ONE instruction of the leader drives both tensor cores -- M = 256 (128 weight rows per CTA), the
            // tile_m tokens of the B operand half in each CTA's shared memory, D in both TMEMs at the same address
            const uint32_t idesc = make_idesc_bf16(pair ? 2 * kTileN : kTileN, tile_m);
            const uint32_t desc_hi = static_cast<uint32_t>(make_smem_desc_sw128(0) >> 32);
            uint32_t stage = 0, phase = 0, astage = 0, aphase = 0;
            unsigned long long wait_ops = 0, wait_acc = 0;
            uint32_t mma_it = 0;  // MMA units so far: picks the accumulator (the epilogue warps count alike)
            for (uint32_t it = 0;; ++it) {
                const uint32_t slot = it % kSchedSlots;
                wait_shared(bar_sfull + 8 * slot, (it / kSchedSlots) & 1, pair);
                const UnitInfo u = ring[slot];
                __syncwarp();  // every lane holds the unit before the slot is handed back
                if (lane == 0) arrive_leader(bar_sempty + 8 * slot, pair);
                if (!u.valid) break;
                if (u.kind == kUnitReduce || !leader) continue;  // (the peer's MMA warp only keeps its ring in step)
                const uint32_t acc = mma_it % acc_stages;
                if (pair) wait_shared(bar_tempty + 8 * acc, ((mma_it / acc_stages) & 1u) ^ 1u, true);
                else mbar_wait_timed(bar_tempty + 8 * acc, ((mma_it / acc_stages) & 1u) ^ 1u, wait_acc);
                ++mma_it;
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + acc * acc_cols;
                for (int kb = u.kb0; kb < u.kb1; ++kb) {
                    if (!unified) mbar_wait_timed(bar_afull + 8 * astage, aphase, wait_ops);
                    mbar_wait_timed(bar_full + 8 * stage, phase, wait_ops);
                    tc_fence_after();
                    if (it == 0 && kb == u.kb0 && lane == 0) my_stats->ts[4] = globaltimer_ns();
                    // operand descriptors: low word = (address >> 4) | LBO field, high word common (ptx.cuh)
                    const uint32_t a_lo = (((smem_base + stage * w_tile_bytes) & 0x3ffffu) >> 4) | (1u << 16);
                    const uint32_t b_lo = (((a_ring + astage * a_tile_bytes) & 0x3ffffu) >> 4) | (1u << 16);
                    if (elect_one()) {
                        // block rr = weight rows [128 rr, 128 rr + 128) of the stage, accumulator columns
                        // [rr tile_m, (rr + 1) tile_m); both blocks read the same activation tile
                        const uint32_t accum = kb > u.kb0 ? 1u : 0u;
                        umma_bf16_kblock<pair>(d_tmem, a_lo, b_lo, desc_hi, idesc, accum);
                        if (!pair && n_sub == 2) umma_bf16_kblock<false>(d_tmem + tile_m, a_lo + (kWTileBytes >> 4), b_lo, desc_hi, idesc, accum);
                        if (pair) {  // the stages of BOTH CTAs are free again
                            umma_commit_pair(bar_empty + 8 * stage);
                            if (!unified) umma_commit_pair(bar_aempty + 8 * astage);
                        } else {
                            umma_commit(bar_empty + 8 * stage);
                            if (!unified) umma_commit(bar_aempty + 8 * astage);
                        }
                        // both CTAs' epilogues drain their own 128 lanes
                        if (kb + 1 == u.kb1) {
                            if (pair) umma_commit_pair(bar_tfull + 8 * acc);
                            else umma_commit(bar_tfull + 8 * acc);
                        }
                    }
                    __syncwarp();
                    if (++stage == static_cast<uint32_t>(stages)) { stage = 0; phase ^= 1; }
                    if (++astage == static_cast<uint32_t>(a_stages)) { astage = 0; aphase ^= 1; }
                }
            }
            if (lane == 0) {
                my_stats->wait[2] = wait_ops;
                my_stats->wait[3] = wait_acc;
            }
        }
    } else {
        // ===== epilogue warps 4..7 (steps a3, a4, a7, a8)
        const int r = threadIdx.x - (kThreads - kEpiThreads);  // TMEM lane = weight row inside a 128-row block
        const int wq = r >> 5;
        unsigned long long wait_acc = 0, wait_part = 0, t_gather = 0, t_partial = 0, t_direct = 0;
        uint32_t mma_it = 0, parity = 0;
        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it % kSchedSlots;
            wait_shared(bar_sfull + 8 * slot, (it / kSchedSlots) & 1, pair);
            const UnitInfo u = ring[slot];
            arrive_leader(bar_sempty + 8 * slot, pair);
            if (!u.valid) break;
            const LayerParams& L = P.layer[u.layer];
            const int m0 = P.m_off + u.m_blk * tile_m;
            const size_t out_row = static_cast<size_t>(L.N);
            const size_t blk_stride = static_cast<size_t>(tile_m) * kTileN;        // floats per 128-row block of a partial
            const size_t ks_stride = blk_stride * n_sub;                           // floats per slice
            // this CTA's 128-row block of the unit: in pair mode the CTAs of a pair own adjacent blocks, and every counter,
            // partial and output column is indexed per 128-row block exactly as without pairing
            const int nblk_c = u.n_blk * nb_mul + static_cast<int>(rank);
            const int ctile = u.m_blk * (L.n_blks * nb_mul) + nblk_c;
            float* const ws_tile = L.ws + static_cast<size_t>(ctile) * L.split * ks_stride;
            bool stored = false;  // this unit wrote (part of) the layer's output
            int red_c0 = 0, red_c1 = 0;  // token columns of the tile whose partials this unit sums (none if equal)
            if (u.kind == kUnitReduce) {
                // ---- step a8, distributed form: sum the partials of token columns [kb0, kb1) of the tile
                if (it < kUnitTrace && r == 0) my_stats->unit_ts[it][2] = globaltimer_ns();
                if (!u.acquired) {
                    if (r == 0)
                        poll_counter(L.arrive + ctile, static_cast<uint32_t>((epoch + 1ull) * static_cast<unsigned long long>(L.split)),
                                     P.status, P.status_host, P.timeout_ns, wait_part);
                    bar_sync(1, kEpiThreads);  // thread 0's acquire happens-before everybody's loads below
                }
                if (r == 0) mbar_arrive(bar_wtaken + 8 * slot);  // late binding: now the scheduler may draw the next ticket
                red_c0 = u.kb0;
                red_c1 = u.kb1;
            } else {
                const uint32_t acc = mma_it % acc_stages;
                const uint32_t taddr = tmem_base + (static_cast<uint32_t>(wq * 32) << 16) + acc * acc_cols;
                mbar_wait_timed(bar_tfull + 8 * acc, (mma_it / acc_stages) & 1u, wait_acc);
                ++mma_it;
                tc_fence_after();
                if (it == 0 && r == 0) my_stats->ts[5] = globaltimer_ns();
                if (it < kUnitTrace && r == 0) my_stats->unit_ts[it][2] = globaltimer_ns();
                const long long te0 = clock64();
                if (L.split == 1) {
                    const EmitCtx e{stage_s, r, L.out, out_row, nblk_c * tile_n, L.N, m0, P.m_end, L.act, tile_m};
                    drain_direct_frag(taddr, static_cast<int>(acc_cols), (bar_tempty + 8 * acc) | (pair ? 1u : 0u), e, parity);
                    stored = true;
                    t_direct += static_cast<unsigned long long>(clock64() - te0);
                } else {
                    // ---- step a8 (split-K): every slice stores its fp32 partial (16-byte pieces, a warp
                    // writes 512 contiguous bytes) and arrives on the tile's counter.
                    // (the columns of the n_sub blocks are consecutive both in TMEM and in the partial)
                    float* wsp = ws_tile + static_cast<size_t>(u.ks) * ks_stride + static_cast<size_t>(r) * 4;
                    const EmitCtx e{};
                    drain_acc<16, false>(taddr, static_cast<int>(acc_cols), (bar_tempty + 8 * acc) | (pair ? 1u : 0u), e, parity, wsp);
                    // the 128 threads' partial stores happen-before thread 0's atomic (bar.sync); its release half
                    // is cumulative and publishes the CTA's whole partial, its acquire half (on the last arrival)
                    // makes the other slices' partials visible to the loads after the second barrier
                    bar_sync(1, kEpiThreads);
                    t_partial += static_cast<unsigned long long>(clock64() - te0);
                    if (L.reduce_mode == kReduceLastArriver) {
                        // whoever arrives LAST sums all partials in fixed slice order and finishes the tile.
                        // Nobody ever waits, so a slow slice delays only its own tile.
                        if (r == 0) {
                            const uint32_t base = static_cast<uint32_t>(epoch * static_cast<unsigned long long>(L.split));
                            const uint32_t old = atom_add_acq_rel_gpu(L.arrive + ctile, 1u) - base;
                            *s_last = (old == static_cast<uint32_t>(L.split - 1)) ? 1u : 0u;
                        }
                        bar_sync(1, kEpiThreads);
                        const bool last = (*s_last != 0);
                        bar_sync(1, kEpiThreads);  // s_last may be rewritten by the next unit only after all have read it
                        if (last) red_c1 = tile_m;
                    } else {
                        // reduce units (their own tickets, later in this layer's table) finish the tile
                        if (r == 0) red_release_gpu_add(L.arrive + ctile, 1u);
                    }
                }
            }
            if (red_c1 > red_c0) {
                const long long tg0 = clock64();
                for (int rr = 0; rr < n_sub; ++rr) {
                    const float* blk = ws_tile + rr * blk_stride;
                    const int n_base = nblk_c * tile_n + rr * kTileN;
                    for (int c = red_c0; c < red_c1; c += 16) {
                        float f[16];
                        uint32_t w[16];
                        gather16(blk, L.split, ks_stride, c, r, f);
#pragma unroll
                        for (int j = 0; j < 16; ++j) w[j] = __float_as_uint(f[j]);
                        emit_cols<16>(w, stage_s, parity, r, L.out, out_row, n_base, L.N, m0 + c, P.m_end, L.act);
                    }
                }
                t_gather += static_cast<unsigned long long>(clock64() - tg0);
                stored = true;
            }
            if (stored && L.publish) {
                // producer epilogue (step a4; output tile, then fence, then the dependency
                // update).  All four epilogue warps wrote the tile: their stores happen-before the
                // barrier, and thread 0's gpu-scope release after it is cumulative (the pattern of a
                // cooperative grid barrier), so one fence + one red publishes the tile -- cf. PAPER.md:129
                // "only the warp responsible for writing global output issues the threadfence".
                fence_proxy_async();  // generic-proxy stores of H vs. the consumers' async-proxy (TMA) reads
                if ((P.flags & kFlagDebugDelay) && u.layer == P.layer_begin) {
                    const uint32_t hsh = (static_cast<uint32_t>(u.tile) * 2654435761u) >> 20;  // 0..4095
                    __nanosleep((hsh & 1023u) * 16u);
                }
                bar_sync(1, kEpiThreads);
                // (test hook MLP_FLAG_DEBUG_DROP_PUBLISH: one producer tile is never published -> its consumers starve -> watchdog)
                const bool drop = (P.flags & kFlagDebugDropPublish) && u.layer == P.layer_begin && ctile == 0;
                if (r == 0 && !drop) red_release_gpu_add(L.ready + ctile, 1u);  // release: orders the tile before the counter
                if (r == 0 && !drop && P.wait_flags && u.layer + 1 < P.layer_end && P.layer[u.layer + 1].use_queue) {
                    // Producer epilogue of the paper's protocol (PAPER.md:95 steps (2)-(4)): look the tile up in the
                    // dependency array, update the scoreboard entry of every group that depends on it, and push the
                    // units of a group whose last dependency this was into the consumer's work queue.
                    const LayerParams& Ln = P.layer[u.layer + 1];
                    const uint32_t tag = static_cast<uint32_t>(epoch + 1ull) & 0xffffu;
                    for (int k = __ldg(Ln.dep_off + u.tile); k < static_cast<int>(__ldg(Ln.dep_off + u.tile + 1)); ++k) {
                        const uint32_t g = __ldg(Ln.dep_list + k);
                        const uint32_t target = static_cast<uint32_t>((epoch + 1ull) * __ldg(Ln.dep_count + g));
                        // acq_rel: releases this tile, and (for the last arrival) acquires every other producer's tile
                        if (atom_add_acq_rel_gpu(Ln.scoreboard + g, 1u) + 1u == target) {
                            const uint32_t base = atom_add_relaxed_gpu(Ln.qtail, static_cast<uint32_t>(Ln.group_units)) -
                                                  static_cast<uint32_t>(epoch * static_cast<unsigned long long>(Ln.units));
                            fence_acq_rel_gpu();  // release pattern for the slot stores below
                            for (int i = 0; i < Ln.group_units; ++i)
                                st_relaxed_gpu(Ln.queue + base + i, (tag << 16) | __ldg(Ln.qorder + g * Ln.group_units + i));
                        }
                    }
                }
            }
            if (it == 0 && r == 0) my_stats->ts[6] = globaltimer_ns();
            if (it < kUnitTrace && r == 0) my_stats->unit_ts[it][3] = globaltimer_ns();
        }
        if (r == 0) {
            my_stats->wait[4] = wait_acc;
            my_stats->wait[5] = wait_part;
            my_stats->wait[1] = t_gather;
            my_stats->wait[6] = t_partial;
            my_stats->wait[7] = t_direct;
        }
    }

    // ------------------------------------------------------------------ teardown
    tc_fence_before();
    if (pair) cluster_sync_all();  // neither CTA leaves (or frees TMEM) while the other may still touch its shared memory / TMEM
    else __syncthreads();
    if (warp == 3) {
        tc_fence_after();
        if (pair) tmem_dealloc_pair(tmem_base, tmem_cols);
        else tmem_dealloc(tmem_base, tmem_cols);
    }
    if (threadIdx.x == 0) {
        my_stats->cycles = static_cast<unsigned long long>(clock64() - t_start);
        my_stats->ts[7] = globaltimer_ns();
        atomicAdd(P.epoch_counter, 1ull);
    }
}

}  // namespace mlp
