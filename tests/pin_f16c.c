/* Test helper (CPU): compares oracle_round16 (integer bit manipulation, oracle/heal_oracle.c)
 * with the x86 F16C hardware conversion VCVTPS2PH (round-to-nearest-even) over ALL 2^32 FP32
 * bit patterns.  NaNs only need to stay NaNs.  Prints "mismatches <n> of 4294967296". */
#include <immintrin.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
uint16_t oracle_round16(float x);
int main(void)
{
    uint64_t bad = 0;
#pragma omp parallel for reduction(+ : bad) schedule(static)
    for (int64_t hi = 0; hi < 65536; ++hi) {
        for (uint32_t lo = 0; lo < 65536; ++lo) {
            uint32_t u = ((uint32_t)hi << 16) | lo;
            float f;
            memcpy(&f, &u, 4);
            uint16_t a = oracle_round16(f);
            uint16_t b = _cvtss_sh(f, _MM_FROUND_TO_NEAREST_INT | _MM_FROUND_NO_EXC);
            if (f != f) bad += !(((a & 0x7c00) == 0x7c00) && (a & 0x3ff));
            else bad += (a != b);
        }
    }
    printf("mismatches %llu of 4294967296\n", (unsigned long long)bad);
    return bad != 0;
}
