// bench_mma_issue.cu -- developer microbenchmark, NOT part of libmlp_pipe.so: what does it cost to ISSUE the tcgen05 work
// of one 64-element K-block (4 MMAs of 128 x N x 16, bf16) from the MMA warp, in SM cycles, against the tensor-core floor of
// 128 N / 256 cycles per MMA?  Operands are resident in shared memory (no loads), the barriers that are waited on are
// already complete, so the figures are pure issue-side cost.  It is the measurement behind the "MMA issuer" paragraph of
// DESIGN.md section 5; its output is profiles/r1d_mma_issue_microbench.txt.
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o /tmp/bench_mma_issue paper_2607_07862_b200/csrc/bench_mma_issue.cu
//   /tmp/bench_mma_issue
//
// Variants (style x waits x commits per K-block):
//   lane0     : the loop runs in ONE thread (`if (lane == 0)`), as the first form of mlp_pipe_kernel did
//   converged : all 32 lanes run the loop and wait, one lane elected with elect.sync issues (the form the kernel uses now)
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "ptx.cuh"
using namespace mlp;

constexpr int kABytes = 16384, kBBytes = 32768;

template <bool kPair>
__device__ __forceinline__ void issue4(uint32_t d, uint64_t a, uint64_t b, uint32_t idesc) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (kPair) umma_bf16_pair(d, a + 2 * k, b + 2 * k, idesc, 1);
        else umma_bf16(d, a + 2 * k, b + 2 * k, idesc, 1);
    }
}
template <bool kPair>
__device__ __forceinline__ void commit1(uint32_t bar) {
    if (kPair) umma_commit_pair(bar);
    else umma_commit(bar);
}

// style 0 = lane0, 1 = converged; n = MMA N; nwait / ncommit per K-block
template <bool kPair>
__global__ void __launch_bounds__(128, 1) issue_kernel(int kblocks, int n, int style, int nwait, int ncommit, unsigned long long* out) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t a_s = base, b_s = base + kABytes, ctrl = b_s + kBBytes;
    const uint32_t bar_done = ctrl, bar_ready = ctrl + 8 /* [2] complete */, bar_sink = ctrl + 24 /* [2] commits land here */, tmem_slot = ctrl + 64;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = kPair ? cluster_ctarank() : 0u;
    for (uint32_t i = threadIdx.x; i < (kABytes + kBBytes) / 4; i += blockDim.x) {  // bf16 values in [1, 2) with random signs
        const uint32_t r = (i * 2654435761u) ^ (blockIdx.x * 40503u);
        const uint32_t v = 0x3f803f80u | (r & 0x007f007fu) | ((r >> 3) & 0x80008000u);
        asm volatile("st.shared.u32 [%0], %1;" ::"r"(base + i * 4), "r"(v));
    }
    fence_proxy_async();
    if (threadIdx.x == 0) {
        for (int i = 0; i < 5; ++i) mbar_init(ctrl + 8 * i, 1);
        fence_mbar_init();
        mbar_arrive(bar_ready);
        mbar_arrive(bar_ready + 8);  // phase 0 of both "operands landed" barriers is complete from the start
    }
    if (warp == 1) {
        if (kPair) { tmem_alloc_pair(tmem_slot, 512); tmem_relinquish_pair(); }
        else { tmem_alloc(tmem_slot, 512); tmem_relinquish(); }
    }
    tc_fence_before();
    __syncthreads();
    if (kPair) cluster_sync_all();
    tc_fence_after();
    uint32_t tmem;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem) : "r"(tmem_slot));
    const uint32_t idesc = make_idesc_bf16(kPair ? 256 : 128, n);
    const uint64_t ad = make_smem_desc_sw128(a_s), bd = make_smem_desc_sw128(b_s);
    if (warp == 0 && rank == 0) {
        if (style == 0) {
            if (lane == 0) {
                const long long t0 = clock64();
                for (int kb = 0; kb < kblocks; ++kb) {
                    for (int w = 0; w < nwait; ++w) mbar_wait(bar_ready + 8 * (w & 1), 0);
                    tc_fence_after();
                    issue4<kPair>(tmem + ((kb & 1) ? n : 0), ad, bd, idesc);
                    for (int c = 0; c < ncommit; ++c) commit1<kPair>(bar_sink + 8 * (c & 1));
                }
                commit1<kPair>(bar_done);
                mbar_wait(bar_done, 0);
                out[blockIdx.x] = static_cast<unsigned long long>(clock64() - t0);
            }
        } else {
            const long long t0 = clock64();
            for (int kb = 0; kb < kblocks; ++kb) {
                for (int w = 0; w < nwait; ++w) mbar_wait(bar_ready + 8 * (w & 1), 0);
                tc_fence_after();
                if (elect_one()) {
                    issue4<kPair>(tmem + ((kb & 1) ? n : 0), ad, bd, idesc);
                    for (int c = 0; c < ncommit; ++c) commit1<kPair>(bar_sink + 8 * (c & 1));
                }
                __syncwarp();
            }
            if (elect_one()) commit1<kPair>(bar_done);
            __syncwarp();
            mbar_wait(bar_done, 0);
            if (lane == 0) out[blockIdx.x] = static_cast<unsigned long long>(clock64() - t0);
        }
    } else if (warp == 0 && kPair) {
        mbar_wait(bar_done, 0);  // (the leader's multicast commit arrives here too)
    }
    __syncthreads();
    if (kPair) cluster_sync_all();
    if (warp == 1) {
        if (kPair) tmem_dealloc_pair(tmem, 512);
        else tmem_dealloc(tmem, 512);
    }
}

template <bool kPair>
static void run(int n, int style, int nwait, int ncommit, unsigned long long* out) {
    const int kblocks = 4096, grid = 148, smem = 1024 + kABytes + kBBytes + 1024;
    cudaFuncSetAttribute(issue_kernel<kPair>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(128);
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = kPair ? 2 : 1;
    at[0].val.clusterDim.y = at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float ms = 0;
    for (int rep = 0; rep < 2; ++rep) {
        cudaMemset(out, 0, grid * sizeof(unsigned long long));
        cudaEventRecord(e0);
        const cudaError_t e = cudaLaunchKernelEx(&cfg, issue_kernel<kPair>, kblocks, n, style, nwait, ncommit, out);
        cudaEventRecord(e1);
        const cudaError_t e2 = cudaDeviceSynchronize();
        if (e != cudaSuccess || e2 != cudaSuccess) {
            printf("error: %s / %s\n", cudaGetErrorString(e), cudaGetErrorString(e2));
            exit(1);
        }
        cudaEventElapsedTime(&ms, e0, e1);
    }
    std::vector<unsigned long long> h(grid);
    cudaMemcpy(h.data(), out, grid * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
    std::vector<double> v;
    for (auto x : h)
        if (x) v.push_back(static_cast<double>(x));
    std::sort(v.begin(), v.end());
    const double cyc = v.empty() ? 0.0 : v[v.size() / 2] / kblocks;
    const double flops = 2.0 * (kPair ? 256 : 128) * n * 64.0 * kblocks * (kPair ? grid / 2 : grid);
    printf("%-5s %-9s N=%3d  waits %d commits %d : %6.1f cycles / K-block (floor %3d)  kernel %7.1f us = %6.0f TFLOP/s\n", kPair ? "pair" : "1-CTA",
           style ? "converged" : "lane0", n, nwait, ncommit, cyc, 4 * 128 * n / 256, ms * 1e3, flops / (ms * 1e-3) / 1e12);
}

int main() {
    unsigned long long* out;
    cudaMalloc(&out, 148 * sizeof(unsigned long long));
    const int ns[3] = {16, 64, 256};
    for (int n : ns) {
        run<false>(n, 0, 0, 0, out);  // bare issue loop
        run<false>(n, 0, 2, 2, out);  // first form of the kernel: two rings, two barriers each
        run<false>(n, 0, 1, 1, out);
        run<false>(n, 1, 2, 2, out);
        run<false>(n, 1, 1, 1, out);  // the kernel now (equally deep rings)
    }
    run<true>(256, 0, 2, 2, out);
    run<true>(256, 1, 1, 1, out);
    cudaFree(out);
    return 0;
}
