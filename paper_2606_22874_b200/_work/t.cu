#include <stdint.h>
__global__ void k(const uint32_t* in, uint32_t* out) {
    uint32_t w = in[threadIdx.x];
    uint32_t r0, r1, r2, r3;
    asm("{ .reg .b8 b0, b1, b2, b3; mov.b32 {b0,b1,b2,b3}, %4; cvt.rn.f16x2.e2m1x2 %0, b0; cvt.rn.f16x2.e2m1x2 %1, b1; cvt.rn.f16x2.e2m1x2 %2, b2; cvt.rn.f16x2.e2m1x2 %3, b3; }"
        : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(w));
    out[threadIdx.x*4] = r0; out[threadIdx.x*4+1] = r1; out[threadIdx.x*4+2] = r2; out[threadIdx.x*4+3] = r3;
}
