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

constexpr int kActNone = 0, kActRelu = 1, kActGeluTanh = 2;
constexpr uint32_t kFlagTileMajor = 0x1u, kFlagDebugDelay = 0x2u, kFlagDebugReverse = 0x4u, kFlagNoEvictFirst = 0x8u;
constexpr uint32_t kStatusFlagTimeout = 1u;

struct LayerParams {
    int K, N;
    int kb_total;  // ceil(K / 64)
    int n_blks;    // ceil(N / 128)
    int split;     // split of the contraction per output tile
    int units;     // n_blks * m_blks * split
    int drawers;   // CTAs that draw tickets of this layer in one launch
    int act;       // activation on this layer's output
    int publish;   // 1 if a later layer consumes this layer's output
    int pad_;
    __nv_bfloat16* out;  // [M x N] row-major
    float* ws;           // split-K partials [tile][split][tile_m][128]
    uint32_t* ticket;    // 1 monotone counter
    uint32_t* arrive;    // [tiles] monotone split-K arrival counters
    uint32_t* ready;     // [tiles] monotone ready counters, tile = m_blk * n_blks + n_blk
};

struct CtaStats {
    unsigned long long stall_cycles;
    unsigned long long polls;
    unsigned long long cycles;
    uint32_t units[kMaxLayers];
};

struct KernelParams {
    CUtensorMap tm_w[kMaxLayers];
    CUtensorMap tm_a[kMaxLayers];  // input activations of layer l: X (l = 0) or H_l
    LayerParams layer[kMaxLayers];
    int layer_begin, layer_end;
    int m_off, m_end;  // token rows [m_off, m_end) of this launch
    int tile_m, m_blks;
    int stages;
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

__global__ void __launch_bounds__(kThreads, 1) mlp_pipe_kernel(const __grid_constant__ KernelParams P) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));

    const int tile_m = P.tile_m;
    const uint32_t a_tile_bytes = static_cast<uint32_t>(tile_m) * (kTileK * 2);
    const uint32_t stage_bytes = kWTileBytes + a_tile_bytes;
    const int stages = P.stages;

    // control block after the stage ring
    uint8_t* ctrl = smem_gen + static_cast<size_t>(stages) * stage_bytes;
    const uint32_t ctrl_s = smem_base + static_cast<uint32_t>(stages) * stage_bytes;
    const uint32_t bar_full = ctrl_s;                          // [kMaxStages]
    const uint32_t bar_empty = bar_full + 8 * kMaxStages;      // [kMaxStages]
    const uint32_t bar_tfull = bar_empty + 8 * kMaxStages;     // [2]
    const uint32_t bar_tempty = bar_tfull + 16;                // [2]
    const uint32_t bar_sfull = bar_tempty + 16;                // [kSchedSlots]
    const uint32_t bar_sempty = bar_sfull + 8 * kSchedSlots;   // [kSchedSlots]
    const uint32_t bar_wtaken = bar_sempty + 8 * kSchedSlots;  // [kSchedSlots]
    constexpr int kBarBytes = 8 * (2 * kMaxStages + 4 + 3 * kSchedSlots);
    UnitInfo* ring = reinterpret_cast<UnitInfo*>(ctrl + kBarBytes);
    volatile uint32_t* s_tmem = reinterpret_cast<volatile uint32_t*>(ctrl + kBarBytes + sizeof(UnitInfo) * kSchedSlots);
    volatile uint32_t* s_last = s_tmem + 1;
    volatile unsigned long long* s_epoch = reinterpret_cast<volatile unsigned long long*>(s_tmem + 2);

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const long long t_start = clock64();

    uint32_t tmem_cols = 32;
    while (tmem_cols < static_cast<uint32_t>(2 * tile_m)) tmem_cols <<= 1;

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
        for (int i = 0; i < 2; ++i) {
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

    // ------------------------------------------------------------------ roles
    if (warp == 0) {
        // ===== scheduler: ticket -> unit (step a1, ordering knob PAPER.md:99-101)
        if (lane == 0) {
            uint32_t done[kMaxLayers];
            for (int l = 0; l < kMaxLayers; ++l) done[l] = 0;
            int l = P.layer_begin;
            if (static_cast<int>(blockIdx.x) >= P.producer_ctas && P.layer_begin + 1 < P.layer_end) l = P.layer_begin + 1;
            uint32_t it = 0;
            bool finished = false;
            while (!finished) {
                UnitInfo u;
                u.valid = 0;
                u.layer = u.m_blk = u.n_blk = u.ks = u.kb0 = u.kb1 = u.tile = 0;
                // claim at most one unit ahead of the W loader (keeps the tail balanced)
                if (it >= 1) mbar_wait(bar_wtaken + 8 * ((it - 1) % kSchedSlots), ((it - 1) / kSchedSlots) & 1);
                while (l < P.layer_end) {
                    const LayerParams& L = P.layer[l];
                    const uint32_t base = static_cast<uint32_t>(epoch * static_cast<unsigned long long>(L.units + L.drawers));
                    uint32_t t = atom_add_relaxed_gpu(L.ticket, 1u) - base;
                    if (t >= static_cast<uint32_t>(L.units)) {
                        ++l;
                        continue;
                    }
                    if ((P.flags & kFlagDebugReverse) && l == P.layer_begin) t = L.units - 1 - t;
                    const int tiles = L.n_blks * P.m_blks;
                    int tile, ks;
                    const bool tile_major = (l == P.layer_begin) || (P.flags & kFlagTileMajor);
                    if (tile_major) {
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
                    u.kb0 = static_cast<int>((static_cast<long long>(ks) * L.kb_total) / L.split);
                    u.kb1 = static_cast<int>((static_cast<long long>(ks + 1) * L.kb_total) / L.split);
                    u.valid = 1;
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
            for (uint32_t it = 0;; ++it) {
                const uint32_t slot = it % kSchedSlots;
                mbar_wait(bar_sfull + 8 * slot, (it / kSchedSlots) & 1);
                const UnitInfo u = ring[slot];
                mbar_arrive(bar_wtaken + 8 * slot);
                mbar_arrive(bar_sempty + 8 * slot);
                if (!u.valid) break;
                const CUtensorMap* tm = &P.tm_w[u.layer];
                for (int kb = u.kb0; kb < u.kb1; ++kb) {
                    mbar_wait(bar_empty + 8 * stage, phase ^ 1);
                    const uint32_t full = bar_full + 8 * stage;
                    mbar_arrive_expect_tx(full, stage_bytes);
                    const uint32_t dst = smem_base + stage * stage_bytes;
                    if (hint) tma_load_2d_hint(dst, tm, kb * kTileK, u.n_blk * kTileN, full, pol);
                    else tma_load_2d(dst, tm, kb * kTileK, u.n_blk * kTileN, full);
                    if (++stage == static_cast<uint32_t>(stages)) { stage = 0; phase ^= 1; }
                }
            }
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
                const bool wait = P.wait_flags && u.layer > P.layer_begin;
                const uint32_t* ready = wait ? P.layer[u.layer - 1].ready + u.m_blk * P.layer[u.layer - 1].n_blks : nullptr;
                int last_slice = -1;
                for (int kb = u.kb0; kb < u.kb1; ++kb) {
                    mbar_wait(bar_empty + 8 * stage, phase ^ 1);
                    if (wait) {
                        const int slice = (kb * kTileK) / kTileN;  // producer tile that wrote these columns
                        if (slice != last_slice) {
                            if (!aborted && static_cast<int32_t>(ld_acquire_gpu(ready + slice) - target) < 0) {
                                const long long c0 = clock64();
                                const uint64_t t0 = globaltimer_ns();
                                uint32_t n = 0;
                                while (static_cast<int32_t>(ld_acquire_gpu(ready + slice) - target) < 0) {
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
                            last_slice = slice;
                            // H was written through the generic proxy; the TMA below reads it through
                            // the async proxy
                            fence_proxy_async();
                        }
                    }
                    const uint32_t dst = smem_base + stage * stage_bytes + kWTileBytes;
                    tma_load_2d(dst, tm, kb * kTileK, P.m_off + u.m_blk * tile_m, bar_full + 8 * stage);
                    if (++stage == static_cast<uint32_t>(stages)) { stage = 0; phase ^= 1; }
                }
            }
            P.stats[blockIdx.x].stall_cycles = stall;
            P.stats[blockIdx.x].polls = polls;
        }
    } else if (warp == 3) {
        // ===== MMA issuer (steps a2, a6)
        if (lane == 0) {
            const uint32_t idesc = make_idesc_bf16(kTileN, tile_m);
            uint32_t stage = 0, phase = 0;
            for (uint32_t it = 0;; ++it) {
                const uint32_t slot = it % kSchedSlots;
                mbar_wait(bar_sfull + 8 * slot, (it / kSchedSlots) & 1);
                const UnitInfo u = ring[slot];
                mbar_arrive(bar_sempty + 8 * slot);
                if (!u.valid) break;
                const uint32_t acc = it & 1u;
                mbar_wait(bar_tempty + 8 * acc, ((it >> 1) & 1u) ^ 1u);
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + acc * static_cast<uint32_t>(tile_m);
                for (int kb = u.kb0; kb < u.kb1; ++kb) {
                    mbar_wait(bar_full + 8 * stage, phase);
                    tc_fence_after();
                    const uint32_t a_addr = smem_base + stage * stage_bytes;
                    const uint32_t b_addr = a_addr + kWTileBytes;
                    const uint64_t a_desc = make_smem_desc_sw128(a_addr);
                    const uint64_t b_desc = make_smem_desc_sw128(b_addr);
#pragma unroll
                    for (int k = 0; k < kTileK / kUmmaK; ++k) {
                        // advancing K by 16 bf16 = 32 B inside the 128 B swizzle span: +2 in the
                        // (addr >> 4) field of the descriptor
                        umma_bf16(d_tmem, a_desc + 2 * k, b_desc + 2 * k, idesc, (kb > u.kb0 || k > 0) ? 1u : 0u);
                    }
                    umma_commit(bar_empty + 8 * stage);
                    if (++stage == static_cast<uint32_t>(stages)) { stage = 0; phase ^= 1; }
                }
                umma_commit(bar_tfull + 8 * acc);
            }
        }
    } else {
        // ===== epilogue warps 4..7 (steps a3, a4, a7, a8)
        const int r = threadIdx.x - (kThreads - kEpiThreads);  // TMEM lane = weight row inside the tile
        const int wq = r >> 5;
        for (uint32_t it = 0;; ++it) {
            const uint32_t slot = it % kSchedSlots;
            mbar_wait(bar_sfull + 8 * slot, (it / kSchedSlots) & 1);
            const UnitInfo u = ring[slot];
            mbar_arrive(bar_sempty + 8 * slot);
            if (!u.valid) break;
            const LayerParams& L = P.layer[u.layer];
            const uint32_t acc = it & 1u;
            mbar_wait(bar_tfull + 8 * acc, (it >> 1) & 1u);
            tc_fence_after();
            const uint32_t taddr = tmem_base + (static_cast<uint32_t>(wq * 32) << 16) + acc * static_cast<uint32_t>(tile_m);
            const int n = u.n_blk * kTileN + r;
            const int m0 = P.m_off + u.m_blk * tile_m;
            const bool n_ok = n < L.N;
            if (L.split == 1) {
                for (int c0 = 0; c0 < tile_m; c0 += 16) {
                    uint32_t v[16];
                    tmem_ld16(taddr + c0, v);
                    tmem_ld_wait();
                    if (c0 + 16 >= tile_m) {  // accumulator fully read: hand TMEM back to the MMA warp
                        tc_fence_before();
                        mbar_arrive(bar_tempty + 8 * acc);
                    }
                    if (n_ok) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) {
                            const int m = m0 + c0 + j;
                            if (m < P.m_end)
                                L.out[static_cast<size_t>(m) * L.N + n] =
                                    __float2bfloat16_rn(act_apply(__uint_as_float(v[j]), L.act));
                        }
                    }
                }
            } else {
                // step a8: fp32 partial to the workspace; the last arriver sums the partials in fixed
                // slice order, so the result does not depend on which CTA arrives last
                float* wsp = L.ws + (static_cast<size_t>(u.tile) * L.split + u.ks) * (static_cast<size_t>(tile_m) * kTileN) + r;
                for (int c0 = 0; c0 < tile_m; c0 += 16) {
                    uint32_t v[16];
                    tmem_ld16(taddr + c0, v);
                    tmem_ld_wait();
                    if (c0 + 16 >= tile_m) {
                        tc_fence_before();
                        mbar_arrive(bar_tempty + 8 * acc);
                    }
#pragma unroll
                    for (int j = 0; j < 16; ++j) wsp[static_cast<size_t>(c0 + j) * kTileN] = __uint_as_float(v[j]);
                }
                __threadfence();
                bar_sync(1, kEpiThreads);
                if (r == 0) {
                    const uint32_t base = static_cast<uint32_t>(epoch * static_cast<unsigned long long>(L.split));
                    const uint32_t old = atom_add_acq_rel_gpu(L.arrive + u.tile, 1u) - base;
                    *s_last = (old == static_cast<uint32_t>(L.split - 1)) ? 1u : 0u;
                }
                bar_sync(1, kEpiThreads);
                const bool last = (*s_last != 0);
                bar_sync(1, kEpiThreads);  // s_last may be rewritten by the next unit only after all have read it
                if (!last) continue;
                __threadfence();
                const float* wsr = L.ws + static_cast<size_t>(u.tile) * L.split * (static_cast<size_t>(tile_m) * kTileN) + r;
                const size_t ks_stride = static_cast<size_t>(tile_m) * kTileN;
                for (int c0 = 0; c0 < tile_m; c0 += 8) {
                    float s[8];
#pragma unroll
                    for (int j = 0; j < 8; ++j) s[j] = ld_cg_f32(wsr + static_cast<size_t>(c0 + j) * kTileN);
                    for (int ks = 1; ks < L.split; ++ks) {
#pragma unroll
                        for (int j = 0; j < 8; ++j)
                            s[j] += ld_cg_f32(wsr + ks * ks_stride + static_cast<size_t>(c0 + j) * kTileN);
                    }
                    if (n_ok) {
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const int m = m0 + c0 + j;
                            if (m < P.m_end)
                                L.out[static_cast<size_t>(m) * L.N + n] = __float2bfloat16_rn(act_apply(s[j], L.act));
                        }
                    }
                }
            }
            if (L.publish) {
                // producer epilogue (step a4; output tile, then fence, then the dependency
                // update -- "only the warp responsible for writing global output issues the threadfence",
                // PAPER.md:129; here all four epilogue warps write, so all fence, then one thread signals)
                __threadfence();
                fence_proxy_async();
                if ((P.flags & kFlagDebugDelay) && u.layer == P.layer_begin) {
                    const uint32_t hsh = (static_cast<uint32_t>(u.tile) * 2654435761u) >> 20;  // 0..4095
                    __nanosleep((hsh & 1023u) * 16u);
                }
                bar_sync(1, kEpiThreads);
                if (r == 0) red_release_gpu_add(L.ready + u.tile, 1u);
            }
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
        P.stats[blockIdx.x].cycles = static_cast<unsigned long long>(clock64() - t_start);
        atomicAdd(P.epoch_counter, 1ull);
    }
}

}  // namespace mlp
