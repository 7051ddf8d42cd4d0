// Independent pin for the oracle's E2M1 / E4M3 rounding (P-2).
// Host-only program: for every bf16 bit pattern prints the code produced by
// NVIDIA's own host conversion routines in cuda_fp4.h / cuda_fp8.h.
// Output: 65536 lines "bits e2m1 e4m3" (hex).  Built by tests with g++.
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <cuda_fp8.h>
#include <cuda_fp4.h>

int main() {
  for (uint32_t b = 0; b < 65536; ++b) {
    uint32_t u = b << 16;
    float f;
    std::memcpy(&f, &u, 4);
    unsigned e2m1 = 0xff, e4m3 = 0xff;
    if (f == f && f - f == 0.0f) {  // finite
      e2m1 = (unsigned)__nv_cvt_float_to_fp4(f, __NV_E2M1, cudaRoundNearest) & 0xf;
      e4m3 = (unsigned)__nv_cvt_float_to_fp8(f, __NV_SATFINITE, __NV_E4M3) & 0xff;
    }
    std::printf("%04x %02x %02x\n", b, e2m1, e4m3);
  }
  return 0;
}
