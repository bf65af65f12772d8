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
//     D         = TMEM, lane = n (128 lanes), column = m (tile_m fp32 columns), double buffered
// so that a decode-sized batch (M = 16) costs a 128 x 16 MMA instead of a padded 128 x 128 one and
// every weight byte is loaded exactly once.
//
// Warp roles (protocol hidden in the scheduler and store warps of a
// warp-specialised persistent kernel):
//     warp 0  scheduler     global atomic ticket -> unit decode -> smem ring (broadcast)   [step a1]
//     warp 1  W loader      TMA loads of weight tiles; never waits on a flag, so W_{l+1} is
//                            prefetched up to the ring depth before A^l exists
//     warp 2  A loader      consumer prologue: ld.acquire.gpu polls the (M-block, K-slice) ready
//                            counter, then TMA-loads the activation tile                    [step a5]
//     warp 3  MMA issuer    tcgen05.mma into TMEM; owns TMEM alloc / dealloc                [a2, a6]
//     warps 4-7 epilogue    tcgen05.ld -> (split-K fix-up) -> act -> bf16 -> global store,
//                            then producer epilogue: fence + red.release.gpu publish        [a3, a4, a7, a8]
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

constexpr int kActNone = 0, kActRelu = 1, kActGeluTanh = 2;
constexpr uint32_t kFlagTileMajor = 0x1u, kFlagDebugDelay = 0x2u, kFlagDebugReverse = 0x4u, kFlagNoEvictFirst = 0x8u;
constexpr uint32_t kStatusFlagTimeout = 1u;

struct LayerParams {
    int K, N;
    int kb_total;  // ceil(K / 64)
    int n_blks;    // ceil(N / 128)
    int split;     // split of the contraction per output tile
    int units;     // n_blks * m_blks * split
    int ticket_inc;  // what one launch adds to the ticket counter: units + CTAs arriving from the layer before
    int ticket_off;  // unit index of the first atomically drawn ticket (= units handed out statically)
    int act;       // activation on this layer's output
    int publish;   // 1 if a later layer consumes this layer's output
    int ks_major;  // unit order: 0 tile-major (slices of a tile adjacent), 1 K-slice-major
    __nv_bfloat16* out;  // [M x N] row-major
    float* ws;           // split-K partials [tile][split][tile_m][128]
    uint32_t* ticket;    // 1 monotone counter
    uint32_t* arrive;    // [tiles] monotone split-K arrival counters
    uint32_t* ready;     // [tiles] monotone ready counters, tile = m_blk * n_blks + n_blk
    const uint16_t* kb_bounds;  // [split + 1] K-block boundaries of the slices (slices may taper)
};

struct CtaStats {
    unsigned long long stall_cycles;
    unsigned long long polls;
    unsigned long long cycles;
    unsigned long long ts[8];  // globaltimer ns: 0 start, 1 setup done, 2 first ticket, 3 first W TMA issued,
                               // 4 first stage landed, 5 first accumulator ready, 6 first unit stored, 7 exit
    unsigned long long wait[6];  // SM cycles blocked: 0 W loader on a free stage, 1 (unused, see stall_cycles),
                                 // 2 MMA on operands, 3 MMA on a free accumulator, 4 epilogue on an accumulator,
                                 // 5 split-K reducer on the other slices' partials
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
    int stages;         // weight ring depth
    int a_stages;       // activation ring depth
    int acc_stages;     // TMEM accumulators in the ring
    int w_group;        // weight K-blocks requested back to back
    int producer_ctas;  // CTAs with blockIdx.x < producer_ctas start at layer_begin, the rest one layer later
    int wait_flags;     // consumer prologue on/off
    uint32_t flags;
    unsigned long long* epoch_counter;  // += 1 per exiting CTA; epoch = value / gridDim.x
    uint32_t* status;
    unsigned long long timeout_ns;
    CtaStats* stats;
};

struct UnitInfo {
    int layer, m_blk, n_blk, ks, kb0, kb1, valid, tile;
    int acquired, pad_[3];  // 1: the scheduler has already seen (and acquired) every ready counter of this unit
};

__device__ __forceinline__ float act_apply(float x, int act) {
    if (act == kActRelu) return x > 0.0f ? x : 0.0f;
    if (act == kActGeluTanh) {
        float u = 0.7978845608028654f * (x + 0.044715f * x * x * x);
        float t;
        asm("tanh.approx.f32 %0, %1;" : "=f"(t) : "f"(u));
        return 0.5f * x * (1.0f + t);
    }
    return x;
}

__device__ __forceinline__ float ld_cg_f32(const float* p) {
    float v;
    asm volatile("ld.global.cg.f32 %0, [%1];" : "=f"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void mbar_wait_timed(uint32_t bar, uint32_t parity, unsigned long long& acc) {
    if (mbar_test(bar, parity)) return;
    const long long t0 = clock64();
    mbar_wait(bar, parity);
    acc += static_cast<unsigned long long>(clock64() - t0);
}

__device__ __forceinline__ void st_cg_f32(float* p, float v) {
    asm volatile("st.global.cg.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory");
}

// Store 16 token columns (rows m_first .. m_first+15 of `out`) of this lane's output feature n as
// bf16 (RNE).  Adjacent lanes hold adjacent n: lane pairs exchange one value per two columns so
// that every lane stores a packed bf16x2 (even lanes the even column, odd lanes the odd one).
__device__ __forceinline__ void store_out16(__nv_bfloat16* out, size_t ld, int n, bool n_ok, int m_first, int m_end,
                                            const float (&f)[16]) {
    const bool odd = (threadIdx.x & 1) != 0;
#pragma unroll
    for (int j = 0; j < 16; j += 2) {
        const uint32_t a = __bfloat16_as_ushort(__float2bfloat16_rn(f[j]));
        const uint32_t b = __bfloat16_as_ushort(__float2bfloat16_rn(f[j + 1]));
        const uint32_t recv = __shfl_xor_sync(0xffffffffu, odd ? a : b, 1);
        const int m = m_first + j + (odd ? 1 : 0);
        const uint32_t packed = odd ? (recv | (b << 16)) : (a | (recv << 16));
        if (n_ok && m < m_end)
            *reinterpret_cast<uint32_t*>(out + static_cast<size_t>(m) * ld + (n & ~1)) = packed;
    }
}

// Spin until *ctr has reached `target` (wrap-safe).  Relaxed polls + one acquire fence = acquire pattern.
// Bounded: after timeout_ns (or when another waiter has already given up) the wait is abandoned, the
// device status word records it, and `true` is returned so that the caller stops waiting for good.
__device__ __forceinline__ bool poll_counter(const uint32_t* ctr, uint32_t target, uint32_t* status,
                                             unsigned long long timeout_ns, unsigned long long& waited) {
    bool gave_up = false;
    if (static_cast<int32_t>(ld_relaxed_gpu(ctr) - target) < 0) {
        const long long c0 = clock64();
        const uint64_t t0 = globaltimer_ns();
        uint32_t n = 0;
        while (static_cast<int32_t>(ld_relaxed_gpu(ctr) - target) < 0) {
            __nanosleep(32);
            if ((++n & 255u) == 0) {
                if (ld_relaxed_gpu(status) != 0) { gave_up = true; break; }
                if (globaltimer_ns() - t0 > timeout_ns) {
                    atomicCAS(status, 0u, kStatusFlagTimeout);
                    gave_up = true;
                    break;
                }
            }
        }
        waited += static_cast<unsigned long long>(clock64() - c0);
    }
    fence_acq_rel_gpu();
    return gave_up;
}

__global__ void __launch_bounds__(kThreads, 1) mlp_pipe_kernel(const __grid_constant__ KernelParams P) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));

    const int tile_m = P.tile_m;
    const uint32_t a_tile_bytes = static_cast<uint32_t>(tile_m) * (kTileK * 2);
    const int stages = P.stages;      // weight ring depth
    const int a_stages = P.a_stages;  // activation ring depth (its own, deeper ring: the consumer prologue's
                                      // polls and fences then run K-blocks ahead of the weight stream)
    const uint32_t a_ring = smem_base + static_cast<uint32_t>(stages) * kWTileBytes;
    const uint32_t ring_bytes = static_cast<uint32_t>(stages) * kWTileBytes + static_cast<uint32_t>(a_stages) * a_tile_bytes;

    // control block after the two rings
    uint8_t* ctrl = smem_gen + ring_bytes;
    const uint32_t ctrl_s = smem_base + ring_bytes;
    const uint32_t bar_full = ctrl_s;                          // [kMaxStages]  weight tile landed
    const uint32_t bar_empty = bar_full + 8 * kMaxStages;      // [kMaxStages]  weight stage consumed
    const uint32_t bar_afull = bar_empty + 8 * kMaxStages;     // [kMaxStages]  activation tile landed
    const uint32_t bar_aempty = bar_afull + 8 * kMaxStages;    // [kMaxStages]  activation stage consumed
    const uint32_t bar_tfull = bar_aempty + 8 * kMaxStages;    // [kMaxAccStages]
    const uint32_t bar_tempty = bar_tfull + 8 * kMaxAccStages;  // [kMaxAccStages]
    const uint32_t bar_sfull = bar_tempty + 8 * kMaxAccStages;  // [kSchedSlots]
    const uint32_t bar_sempty = bar_sfull + 8 * kSchedSlots;   // [kSchedSlots]
    const uint32_t bar_wtaken = bar_sempty + 8 * kSchedSlots;  // [kSchedSlots]
    constexpr int kBarBytes = 8 * (4 * kMaxStages + 2 * kMaxAccStages + 3 * kSchedSlots);
    UnitInfo* ring = reinterpret_cast<UnitInfo*>(ctrl + kBarBytes);
    volatile uint32_t* s_tmem = reinterpret_cast<volatile uint32_t*>(ctrl + kBarBytes + sizeof(UnitInfo) * kSchedSlots);
    volatile uint32_t* s_last = s_tmem + 1;
    volatile unsigned long long* s_epoch = reinterpret_cast<volatile unsigned long long*>(s_tmem + 2);

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const long long t_start = clock64();
    CtaStats* const my_stats = P.stats + blockIdx.x;
    if (threadIdx.x == 0) my_stats->ts[0] = globaltimer_ns();

    // TMEM accumulator ring: as many tile_m-column accumulators as fit (<= 8), so that the MMA warp can
    // run ahead of an epilogue that is waiting on a memory round trip
    const uint32_t acc_stages = static_cast<uint32_t>(P.acc_stages);
    uint32_t tmem_cols = 32;
    while (tmem_cols < acc_stages * static_cast<uint32_t>(tile_m)) tmem_cols <<= 1;

    // ------------------------------------------------------------------ one-time setup
    if (threadIdx.x == 0) {
        // device-resident epoch: no per-run host state, so a captured graph can be replayed
        *s_epoch = ld_relaxed_gpu_u64(reinterpret_cast<const uint64_t*>(P.epoch_counter)) / gridDim.x;
        for (int l = P.layer_begin; l < P.layer_end; ++l) {
            prefetch_tmap(&P.tm_w[l]);
            prefetch_tmap(&P.tm_a[l]);
        }
    }
    if (threadIdx.x == 32) {
        for (int s = 0; s < stages; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, 1);
        }
        for (int s = 0; s < a_stages; ++s) {
            mbar_init(bar_afull + 8 * s, 1);
            mbar_init(bar_aempty + 8 * s, 1);
        }
        for (int i = 0; i < kMaxAccStages; ++i) {
            mbar_init(bar_tfull + 8 * i, 1);
            mbar_init(bar_tempty + 8 * i, kEpiThreads);
        }
        for (int i = 0; i < kSchedSlots; ++i) {
            mbar_init(bar_sfull + 8 * i, 1);
            mbar_init(bar_sempty + 8 * i, 3 + kEpiThreads);
            mbar_init(bar_wtaken + 8 * i, 1);
        }
        fence_mbar_init();
    }
    if (warp == 3) {
        tmem_alloc(smem_u32(const_cast<uint32_t*>(s_tmem)), tmem_cols);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *s_tmem;
    const unsigned long long epoch = *s_epoch;
    if (threadIdx.x == 0) my_stats->ts[1] = globaltimer_ns();

    // ------------------------------------------------------------------ roles
    if (warp == 0) {
        // ===== scheduler: ticket -> unit (step a1, ordering knob PAPER.md:99-101)
        if (lane == 0) {
            uint32_t done[kMaxLayers];
            for (int l = 0; l < kMaxLayers; ++l) done[l] = 0;
            int l = P.layer_begin;
            // the first unit of a CTA is static (its rank among the CTAs that start on the same layer):
            // no atomic round trip before the first weight load
            uint32_t static_id = blockIdx.x;
            bool use_static = true;
            if (static_cast<int>(blockIdx.x) >= P.producer_ctas && P.layer_begin + 1 < P.layer_end) {
                l = P.layer_begin + 1;
                static_id = blockIdx.x - P.producer_ctas;
            }
            uint32_t it = 0;
            bool finished = false;
            while (!finished) {
                UnitInfo u;
                u.valid = 0;
                u.layer = u.m_blk = u.n_blk = u.ks = u.kb0 = u.kb1 = u.tile = u.acquired = 0;
                // claim at most one unit ahead of the W loader (keeps the tail balanced)
                if (it >= 1) mbar_wait(bar_wtaken + 8 * ((it - 1) % kSchedSlots), ((it - 1) / kSchedSlots) & 1);
                while (l < P.layer_end) {
                    const LayerParams& L = P.layer[l];
                    uint32_t t;
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
                    if ((P.flags & kFlagDebugReverse) && l == P.layer_begin) t = L.units - 1 - t;
                    const int tiles = L.n_blks * P.m_blks;
                    int tile, ks;
                    if (!L.ks_major) {
                        tile = t / L.split;
                        ks = t % L.split;
                    } else {  // K-slice-major: early units depend on early producer tiles only
                        ks = t / tiles;
                        tile = t % tiles;
                    }
                    u.layer = l;
                    u.tile = tile;
                    u.m_blk = tile / L.n_blks;
                    u.n_blk = tile % L.n_blks;
                    u.ks = ks;
                    u.kb0 = __ldg(L.kb_bounds + ks);
                    u.kb1 = __ldg(L.kb_bounds + ks + 1);
                    u.valid = 1;
                    if (P.wait_flags && l > P.layer_begin && !(P.flags & 0x80u)) {
                        // Consumer prologue, fast path (the prologue lives in the scheduler
                        // warp): one look at all ready counters under this unit's K range.  If every producer
                        // tile is already published -- the normal case, the scheduler runs a unit ahead --
                        // ONE acquire fence here covers the whole unit and the loaders never poll.  Otherwise
                        // the activation loader polls slice by slice while the weight loader prefetches.
                        const uint32_t target = static_cast<uint32_t>(epoch + 1ull);
                        const uint32_t* rd = P.layer[l - 1].ready + u.m_blk * P.layer[l - 1].n_blks;
                        const int s0 = (u.kb0 * kTileK) / kTileN, s1 = ((u.kb1 - 1) * kTileK) / kTileN + 1;
                        bool all = (s1 - s0) <= 32;
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
                if (it >= kSchedSlots) mbar_wait(bar_sempty + 8 * slot, ((it / kSchedSlots) & 1) ^ 1);
                ring[slot] = u;
                mbar_arrive(bar_sfull + 8 * slot);  // release: ring[slot] visible to waiters
                ++it;
            }
            for (int l2 = 0; l2 < kMaxLayers; ++l2) P.stats[blockIdx.x].units[l2] = done[l2];
        }
    } else if (warp == 1) {
        // ===== W loader
        if (lane == 0) {
            const uint64_t pol = policy_evict_first();
            const bool hint = !(P.flags & kFlagNoEvictFirst);
            uint32_t stage = 0, phase = 0;
            unsigned long long w_wait = 0;
            for (uint32_t it = 0;; ++it) {
                const uint32_t slot = it % kSchedSlots;
                mbar_wait(bar_sfull + 8 * slot, (it / kSchedSlots) & 1);
                const UnitInfo u = ring[slot];
                mbar_arrive(bar_wtaken + 8 * slot);
                mbar_arrive(bar_sempty + 8 * slot);
                if (!u.valid) break;
                if (it < kUnitTrace) {
                    my_stats->unit_ts[it][0] = globaltimer_ns();
                    my_stats->unit_id[it] = (static_cast<uint32_t>(u.layer) << 28) | (static_cast<uint32_t>(u.tile) << 8) | static_cast<uint32_t>(u.ks);
                }
                const CUtensorMap* tm = &P.tm_w[u.layer];
                // K-blocks are requested in groups of w_group: the loader first waits until the whole group of
                // stages is free and then issues the group back to back, so that the 128-byte pieces of one
                // weight row that are adjacent in memory reach the DRAM controller together
                for (int kb = u.kb0; kb < u.kb1;) {
                    const int g = min(P.w_group, u.kb1 - kb);
                    uint32_t st = stage, ph = phase;
                    for (int i = 0; i < g; ++i) {
                        mbar_wait_timed(bar_empty + 8 * st, ph ^ 1, w_wait);
                        if (++st == static_cast<uint32_t>(stages)) { st = 0; ph ^= 1; }
                    }
                    for (int i = 0; i < g; ++i, ++kb) {
                        const uint32_t full = bar_full + 8 * stage;
                        mbar_arrive_expect_tx(full, kWTileBytes);
                        const uint32_t dst = smem_base + stage * kWTileBytes;
                        if (hint) tma_load_2d_hint(dst, tm, kb * kTileK, u.n_blk * kTileN, full, pol);
                        else tma_load_2d(dst, tm, kb * kTileK, u.n_blk * kTileN, full);
                        if (it == 0 && kb == u.kb0) my_stats->ts[3] = globaltimer_ns();
                        if (++stage == static_cast<uint32_t>(stages)) { stage = 0; phase ^= 1; }
                    }
                }
                if (it < kUnitTrace) my_stats->unit_ts[it][1] = globaltimer_ns();
            }
            my_stats->wait[0] = w_wait;
        }
    } else if (warp == 2) {
        // ===== A loader = consumer prologue (step a5; PAPER.md:95 step (5))
        if (lane == 0) {
            uint32_t stage = 0, phase = 0;
            unsigned long long stall = 0, polls = 0;
            bool aborted = false;
            const uint32_t target = static_cast<uint32_t>(epoch + 1ull);
            for (uint32_t it = 0;; ++it) {
                const uint32_t slot = it % kSchedSlots;
                mbar_wait(bar_sfull + 8 * slot, (it / kSchedSlots) & 1);
                const UnitInfo u = ring[slot];
                mbar_arrive(bar_sempty + 8 * slot);
                if (!u.valid) break;
                const CUtensorMap* tm = &P.tm_a[u.layer];
                const bool wait = P.wait_flags && u.layer > P.layer_begin && !u.acquired;
                if (P.wait_flags && u.layer > P.layer_begin) fence_proxy_async();
                const uint32_t* ready = wait ? P.layer[u.layer - 1].ready + u.m_blk * P.layer[u.layer - 1].n_blks : nullptr;
                // Slices [.., ready_upto) of this unit are known to be published.  Readiness is monotone
                // within a run, so the prologue looks ahead: up to 8 counters are read with independent
                // relaxed loads that are ISSUED a few K-blocks before their result is needed (the round trip
                // overlaps the TMA issue of slices already known to be ready), then one acquire fence turns
                // the observations into an acquire pattern (PTX memory model: relaxed read + fence.acq_rel).
                const int slice_end = wait ? ((u.kb1 - 1) * kTileK) / kTileN + 1 : 0;
                int ready_upto = wait ? (u.kb0 * kTileK) / kTileN : 0;
                uint32_t v[8];
                int pend_base = -1;  // >= 0: v[] holds in-flight reads of counters pend_base .. pend_base+7
                for (int kb = u.kb0; kb < u.kb1; ++kb) {
                    mbar_wait(bar_aempty + 8 * stage, phase ^ 1);
                    if (wait) {
                        const int slice = (kb * kTileK) / kTileN;  // producer tile that wrote these columns
                        if (pend_base < 0 && ready_upto < slice_end && slice + 2 >= ready_upto) {
                            pend_base = ready_upto;
#pragma unroll
                            for (int i = 0; i < 8; ++i)
                                v[i] = (pend_base + i < slice_end) ? ((P.flags & 0x40u) ? ld_acquire_gpu(ready + pend_base + i) : ld_relaxed_gpu(ready + pend_base + i)) : target - 1u;
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
                                    while (static_cast<int32_t>(ld_relaxed_gpu(ready + slice) - target) < 0) {
                                        ++n;
                                        __nanosleep(32);
                                        if ((n & 255u) == 0) {
                                            if (ld_relaxed_gpu(P.status) != 0) { aborted = true; break; }
                                            if (globaltimer_ns() - t0 > P.timeout_ns) {
                                                atomicCAS(P.status, 0u, kStatusFlagTimeout);
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
                            if (!(P.flags & 0x10u)) fence_acq_rel_gpu();
                            // H was written through the generic proxy; the TMA below reads it through
                            // the async proxy
                            if (!(P.flags & 0x20u)) fence_proxy_async();
                            ready_upto = pend_base + n_ok;
                            pend_base = -1;
                        }
                    }
                    mbar_arrive_expect_tx(bar_afull + 8 * stage, a_tile_bytes);
                    tma_load_2d(a_ring + stage * a_tile_bytes, tm, kb * kTileK, P.m_off + u.m_blk * tile_m, bar_afull + 8 * stage);
                    if (++stage == static_cast<uint32_t>(a_stages)) { stage = 0; phase ^= 1; }
                }
            }
            P.stats[blockIdx.x].stall_cycles = stall;
            P.stats[blockIdx.x].polls = polls;
        }
    } else if (warp == 3) {
        // ===== MMA issuer (steps a2, a6)
        if (lane == 0) {
            const uint32_t idesc = make_idesc_bf16(kTileN, tile_m);
            uint32_t stage = 0, phase = 0, astage = 0, aphase = 0;
            unsigned long long wait_ops = 0, wait_acc = 0;
            for (uint32_t it = 0;; ++it) {
                const uint32_t slot = it % kSchedSlots;
                mbar_wait(bar_sfull + 8 * slot, (it / kSchedSlots) & 1);
                const UnitInfo u = ring[slot];
                mbar_arrive(bar_sempty + 8 * slot);
                if (!u.valid) break;
                const uint32_t acc = it % acc_stages;
                mbar_wait_timed(bar_tempty + 8 * acc, ((it / acc_stages) & 1u) ^ 1u, wait_acc);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + acc * static_cast<uint32_t>(tile_m);
                for (int kb = u.kb0; kb < u.kb1; ++kb) {
                    mbar_wait_timed(bar_afull + 8 * astage, aphase, wait_ops);
                    mbar_wait_timed(bar_full + 8 * stage, phase, wait_ops);
                    tc_fence_after();
                    if (it == 0 && kb == u.kb0) my_stats->ts[4] = globaltimer_ns();
                    const uint32_t a_addr = smem_base + stage * kWTileBytes;
                    const uint32_t b_addr = a_ring + astage * a_tile_bytes;
                    const uint64_t a_desc = make_smem_desc_sw128(a_addr);
                    const uint64_t b_desc = make_smem_desc_sw128(b_addr);
#pragma unroll
                    for (int k = 0; k < kTileK / kUmmaK; ++k) {
                        // advancing K by 16 bf16 = 32 B inside the 128 B swizzle span: +2 in the
                        // (addr >> 4) field of the descriptor
                        umma_bf16(d_tmem, a_desc + 2 * k, b_desc + 2 * k, idesc, (kb > u.kb0 || k > 0) ? 1u : 0u);
                    }
                    umma_commit(bar_empty + 8 * stage);
                    umma_commit(bar_aempty + 8 * astage);
                    if (++stage == static_cast<uint32_t>(stages)) { stage = 0; phase ^= 1; }
                    if (++astage == static_cast<uint32_t>(a_stages)) { astage = 0; aphase ^= 1; }
                }
                umma_commit(bar_tfull + 8 * acc);
            }
            my_stats->wait[2] = wait_ops;
            my_stats->wait[3] = wait_acc;
        }
    } else {
        // ===== epilogue warps 4..7 (steps a3, a4, a7, a8)
        const int r = threadIdx.x - (kThreads - kEpiThreads);  // TMEM lane = weight row inside the tile
        const int wq = r >> 5;
        unsigned long long wait_acc = 0, wait_part = 0;
        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it % kSchedSlots;
            mbar_wait(bar_sfull + 8 * slot, (it / kSchedSlots) & 1);
            const UnitInfo u = ring[slot];
            mbar_arrive(bar_sempty + 8 * slot);
            if (!u.valid) break;
            const LayerParams& L = P.layer[u.layer];
            const uint32_t acc = it % acc_stages;
            const uint32_t taddr = tmem_base + (static_cast<uint32_t>(wq * 32) << 16) + acc * static_cast<uint32_t>(tile_m);
            const int n = u.n_blk * kTileN + r;
            const int m0 = P.m_off + u.m_blk * tile_m;
            const bool n_ok = n < L.N;
            const size_t out_row = static_cast<size_t>(L.N);
            const size_t ks_stride = static_cast<size_t>(tile_m) * kTileN;
            float* const ws_tile = L.ws + static_cast<size_t>(u.tile) * L.split * ks_stride + r;
            mbar_wait_timed(bar_tfull + 8 * acc, (it / acc_stages) & 1u, wait_acc);
            tc_fence_after();
            if (it == 0 && r == 0) my_stats->ts[5] = globaltimer_ns();
            if (it < kUnitTrace && r == 0) my_stats->unit_ts[it][2] = globaltimer_ns();
            if (L.split == 1) {
                for (int c0 = 0; c0 < tile_m; c0 += 16) {
                    uint32_t v[16];
                    tmem_ld16(taddr + c0, v);
                    tmem_ld_wait();
                    if (c0 + 16 >= tile_m) {  // accumulator fully read: hand TMEM back to the MMA warp
                        tc_fence_before();
                        mbar_arrive(bar_tempty + 8 * acc);
                    }
                    float sum[16];
#pragma unroll
                    for (int j = 0; j < 16; ++j) sum[j] = act_apply(__uint_as_float(v[j]), L.act);
                    store_out16(L.out, out_row, n, n_ok, m0 + c0, P.m_end, sum);
                }
            } else {
                // ---- step a8 (split-K): every slice stores its fp32 partial and arrives on the tile's counter;
                // whoever arrives LAST sums all partials in fixed slice order (so the rounding does not depend
                // on who that is) and finishes the tile.  Nobody ever waits, so a slow slice delays only its
                // own tile, never the epilogue warps of another CTA.
                float* wsp = ws_tile + static_cast<size_t>(u.ks) * ks_stride;
                for (int c0 = 0; c0 < tile_m; c0 += 16) {
                    uint32_t v[16];
                    tmem_ld16(taddr + c0, v);
                    tmem_ld_wait();
                    if (c0 + 16 >= tile_m) {
                        tc_fence_before();
                        mbar_arrive(bar_tempty + 8 * acc);
                    }
#pragma unroll
                    for (int j = 0; j < 16; ++j) st_cg_f32(wsp + static_cast<size_t>(c0 + j) * kTileN, __uint_as_float(v[j]));
                }
                // the 128 threads' partial stores happen-before thread 0's atomic (bar.sync); its release half
                // is cumulative and publishes the CTA's whole partial, its acquire half (on the last arrival)
                // makes the other slices' partials visible to the loads after the second barrier
                bar_sync(1, kEpiThreads);
                if (r == 0) {
                    const uint32_t base = static_cast<uint32_t>(epoch * static_cast<unsigned long long>(L.split));
                    const uint32_t old = atom_add_acq_rel_gpu(L.arrive + u.tile, 1u) - base;
                    *s_last = (old == static_cast<uint32_t>(L.split - 1)) ? 1u : 0u;
                }
                bar_sync(1, kEpiThreads);
                const bool last = (*s_last != 0);
                bar_sync(1, kEpiThreads);  // s_last may be rewritten by the next unit only after all have read it
                if (!last) {
                    if (it < kUnitTrace && r == 0) my_stats->unit_ts[it][3] = globaltimer_ns();
                    continue;
                }
                for (int c0 = 0; c0 < tile_m; c0 += 16) {
                    float sum[16];
                    // up to 16 * kGather independent loads in flight per thread; the adds stay in slice order
                    for (int ks = 0; ks < L.split; ks += kGather) {
                        float t[kGather][16];
#pragma unroll
                        for (int q = 0; q < kGather; ++q)
                            if (ks + q < L.split) {
#pragma unroll
                                for (int j = 0; j < 16; ++j)
                                    t[q][j] = ld_cg_f32(ws_tile + (ks + q) * ks_stride + static_cast<size_t>(c0 + j) * kTileN);
                            }
#pragma unroll
                        for (int q = 0; q < kGather; ++q)
                            if (ks + q < L.split) {
                                if (ks + q == 0) {
#pragma unroll
                                    for (int j = 0; j < 16; ++j) sum[j] = t[q][j];
                                } else {
#pragma unroll
                                    for (int j = 0; j < 16; ++j) sum[j] += t[q][j];
                                }
                            }
                    }
#pragma unroll
                    for (int j = 0; j < 16; ++j) sum[j] = act_apply(sum[j], L.act);
                    store_out16(L.out, out_row, n, n_ok, m0 + c0, P.m_end, sum);
                }
            }
            if (L.publish) {
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
                if (r == 0) red_release_gpu_add(L.ready + u.tile, 1u);  // release: orders the tile before the counter
            }
            if (it == 0 && r == 0) my_stats->ts[6] = globaltimer_ns();
            if (it < kUnitTrace && r == 0) my_stats->unit_ts[it][3] = globaltimer_ns();
        }
        if (r == 0) {
            my_stats->wait[4] = wait_acc;
            my_stats->wait[5] = wait_part;
        }
    }

    // ------------------------------------------------------------------ teardown
    tc_fence_before();
    __syncthreads();
    if (warp == 3) {
        tc_fence_after();
        tmem_dealloc(tmem_base, tmem_cols);
    }
    if (threadIdx.x == 0) {
        my_stats->cycles = static_cast<unsigned long long>(clock64() - t_start);
        my_stats->ts[7] = globaltimer_ns();
        atomicAdd(P.epoch_counter, 1ull);
    }
}

}  // namespace mlp
