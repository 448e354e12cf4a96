/* Third, independent CRC32C: the x86 SSE4.2 crc32 instruction (tests only). */
#include <stdint.h>
#include <nmmintrin.h>
uint32_t hw_crc32c(const uint8_t *p, uint64_t n) {
    uint32_t c = 0xFFFFFFFFu;
    for (uint64_t i = 0; i < n; i++) c = _mm_crc32_u8(c, p[i]);
    return c ^ 0xFFFFFFFFu;
}
