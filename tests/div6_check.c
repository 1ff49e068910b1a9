/* Check of an arithmetic fact the fp32 convdiff kernel relies on (csrc/wl_convdiff.cuh, cd_div6): for finite x with
 * |x| >= 2^-100,  q = RN(x * RN(1/6)),  r = fma(-6, q, x),  q' = fma(r, RN(1/6), q)  equals the IEEE quotient RN(x / 6).
 * IEEE arithmetic is the same on the host and on the device, so the host can check it exhaustively.
 * usage: div6_check <first bit pattern> <count>; prints the number of finite x in range whose q' differs from x / 6. */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

int main(int argc, char** argv) {
    const uint64_t first = strtoull(argv[1], 0, 0), count = strtoull(argv[2], 0, 0);
    const float y = 1.0f / 6.0f;
    uint64_t bad = 0;
    for (uint64_t b = first; b < first + count; ++b) {
        const uint32_t u = (uint32_t)b;
        float x;
        memcpy(&x, &u, 4);
        if (isnan(x) || isinf(x) || !(fabsf(x) >= 0x1p-100f)) continue;
        volatile float q = x * y;
        const float r = fmaf(-6.0f, q, x);
        const float q2 = fmaf(r, y, q);
        const float ref = x / 6.0f;
        if (memcmp(&q2, &ref, 4) != 0) ++bad;
    }
    printf("%llu\n", (unsigned long long)bad);
    return 0;
}
