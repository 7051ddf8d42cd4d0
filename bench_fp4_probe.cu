// bench_fp4_probe.cu -- measurement only, built and run by bench.py: the rate of
// tcgen05.mma.cta_group::2.kind::mxf4nvf4.block_scale (M=256, N=256, K=64) with operands fixed in shared memory,
// the accumulator in TMEM and nothing else in the loop (no TMA, no epilogue); optionally with the 12 tcgen05.cp
// scale copies the GEMM issues per K=256 stage.  Not part of the library (it only borrows the PTX wrappers of
// paper_2607_05711_b200/csrc/common.cuh).
//   bench_fp4_probe [iterations]            the round-1 table: 1 / 4 operand stages x with / without scale copies
//   bench_fp4_probe --sustained SECONDS     all CTA pairs, 4 stages, scale copies on, back-to-back launches for
//                                           SECONDS; prints one line "sustained ... TFLOP/s" (the FP4 ceiling
//                                           under the power cap, next to which bench.py samples the SM clock)
// Round 1 on B200: exactly 128.0 cycles per MMA in every variant, 8.3-8.4 PFLOP/s chip-wide over a 1.2 ms burst.
#include <cstdio>
#include <cstdlib>
#include <vector>
#include <cstring>
#include <chrono>
#include "paper_2607_05711_b200/csrc/common.cuh"
using namespace ft;
thread_local int ft::g_last_cuda_error = 0;

constexpr int A_BYTES = 128 * 128, B_BYTES = 128 * 128, SF_BYTES = 2048 + 4096;
constexpr int STAGE = A_BYTES + B_BYTES + SF_BYTES;

// mode 0: MMA only; mode 1: + 12 tcgen05.cp per 4 MMAs; mode 2: cta_group::1 M=128 N=256 (single CTA)
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(128, 1)
k_probe(int iters, int mode, int nstages, long long* out) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  __shared__ uint64_t done_bar;
  __shared__ uint32_t tmem_base_s;
  const int warp = threadIdx.x >> 5;
  const uint32_t rank = cluster_ctarank();
  // fill smem with a pattern (valid e2m1 codes = any bits; scales: 0x38 = 1.0)
  for (int i = threadIdx.x; i < nstages * STAGE / 4; i += 128) {
    uint32_t v = 0x12345678u * (i + 1) + rank;
    reinterpret_cast<uint32_t*>(smem)[i] = v;
  }
  __syncthreads();
  for (int s = 0; s < nstages; ++s)
    for (int i = threadIdx.x; i < SF_BYTES / 4; i += 128)
      reinterpret_cast<uint32_t*>(smem + s * STAGE + A_BYTES + B_BYTES)[i] = 0x38383838u;
  if (threadIdx.x == 0) { mbar_init(&done_bar, 1); fence_mbar_init(); }
  if (warp == 2) { tmem_alloc2(&tmem_base_s, 512); tmem_relinquish2(); }
  fence_proxy_async();
  tc_fence_before();
  cluster_sync();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;
  if (warp == 1 && rank == 0 && elect_one()) {
    constexpr uint32_t idesc4 = idesc_nvf4(256, 256);
    const uint32_t sfa_t = tmem_base + 256, sfb_t = tmem_base + 256 + 16;
    // scales once
    {
      const uint32_t ssfa = smem_u32(smem) + A_BYTES + B_BYTES, ssfb = ssfa + 2048;
      for (int k = 0; k < 4; ++k) {
        tc_cp_sf_pair(sfa_t + 4 * k, make_smem_desc(ssfa + k * 512, 128, 0, 0));
        tc_cp_sf_pair(sfb_t + 8 * k, make_smem_desc(ssfb + k * 512, 128, 0, 0));
        tc_cp_sf_pair(sfb_t + 8 * k + 4, make_smem_desc(ssfb + 2048 + k * 512, 128, 0, 0));
      }
    }
    const long long t0 = clock64();
    int st = 0;
    for (int it = 0; it < iters; ++it) {
      const uint32_t sa = smem_u32(smem + st * STAGE), sb = sa + A_BYTES;
      if (mode == 1) {
        const uint32_t ssfa = sb + B_BYTES, ssfb = ssfa + 2048;
        for (int k = 0; k < 4; ++k) {
          tc_cp_sf_pair(sfa_t + 4 * k, make_smem_desc(ssfa + k * 512, 128, 0, 0));
          tc_cp_sf_pair(sfb_t + 8 * k, make_smem_desc(ssfb + k * 512, 128, 0, 0));
          tc_cp_sf_pair(sfb_t + 8 * k + 4, make_smem_desc(ssfb + 2048 + k * 512, 128, 0, 0));
        }
      }
      for (int k = 0; k < 4; ++k)
        mma_nvf4_pair(tmem_base, make_smem_desc(sa + k * 32, 1024, 0, 2), make_smem_desc(sb + k * 32, 1024, 0, 2),
                      idesc4, sfa_t + 4 * k, sfb_t + 8 * k, (it | k) != 0);
      if (++st == nstages) st = 0;
    }
    tc_commit_pair(&done_bar, 1);
    mbar_wait(&done_bar, 0);
    const long long t1 = clock64();
    out[blockIdx.x >> 1] = t1 - t0;
  }
  tc_fence_before();
  cluster_sync();
  if (warp == 2) { tc_fence_after(); tmem_dealloc2(tmem_base, 512); }
}

int main(int argc, char** argv) {
  int nsm = 0;
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, 0);
  long long* d;
  cudaMalloc(&d, 1024 * 8);
  if (argc > 2 && strcmp(argv[1], "--sustained") == 0) {
    const double seconds = atof(argv[2]);
    const int nstages = 4, mode = 1, iters = 20000;   // ~5 ms per launch
    const int smem = nstages * STAGE + 1024;
    cudaFuncSetAttribute(k_probe, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    cudaMemset(d, 0, 1024 * 8);
    k_probe<<<nsm, 128, smem>>>(iters, mode, nstages, d);   // warm
    cudaDeviceSynchronize();
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const auto t0 = std::chrono::steady_clock::now();
    long launches = 0;
    cudaEventRecord(e0);
    do {
      for (int i = 0; i < 8; ++i) k_probe<<<nsm, 128, smem>>>(iters, mode, nstages, d);
      launches += 8;
      cudaStreamSynchronize(0);
    } while (std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count() < seconds);
    cudaEventRecord(e1);
    cudaError_t e = cudaDeviceSynchronize();
    float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
    std::vector<long long> h(nsm / 2);
    cudaMemcpy(h.data(), d, nsm / 2 * 8, cudaMemcpyDeviceToHost);
    double cyc = 0; for (auto v : h) cyc += (double)v; cyc /= (nsm / 2);
    const double flop = 2.0 * 256 * 256 * 64 * 4.0 * iters * (nsm / 2) * launches;
    printf("sustained %s %.3f s %ld launches: %.1f cycles per MMA (last launch), %.0f TFLOP/s\n", cudaGetErrorString(e),
           ms * 1e-3, launches, cyc / (4.0 * iters), flop / (ms * 1e-3) / 1e12);
    return e == cudaSuccess ? 0 : 1;
  }
  const int iters = argc > 1 ? atoi(argv[1]) : 2000;
  for (int nstages : {1, 4})
    for (int mode : {0, 1}) {
      const int smem = nstages * STAGE + 1024;
      cudaFuncSetAttribute(k_probe, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
      for (int grid : {2, nsm}) {
        cudaMemset(d, 0, 1024 * 8);
        cudaEvent_t e0, e1;
        cudaEventCreate(&e0); cudaEventCreate(&e1);
        k_probe<<<grid, 128, smem>>>(iters, mode, nstages, d);   // warm
        cudaEventRecord(e0);
        k_probe<<<grid, 128, smem>>>(iters, mode, nstages, d);
        cudaEventRecord(e1);
        cudaError_t e = cudaDeviceSynchronize();
        float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
        std::vector<long long> h(grid / 2);
        cudaMemcpy(h.data(), d, grid / 2 * 8, cudaMemcpyDeviceToHost);
        double cyc = 0; for (auto v : h) cyc += (double)v; cyc /= (grid / 2);
        const double mma = 4.0 * iters;
        const double flop = 2.0 * 256 * 256 * 64 * mma * (grid / 2);
        printf("stages %d mode %d grid %3d: %s  %.1f cycles per MMA (M256 N256 K64), %.0f TFLOP/s by events (%.3f ms)\n",
               nstages, mode, grid, cudaGetErrorString(e), cyc / mma, flop / (ms * 1e-3) / 1e12, ms);
      }
    }
  return 0;
}
