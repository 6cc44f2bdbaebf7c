/* tests/asan_driver.c — the CPU oracle under AddressSanitizer + UndefinedBehaviorSanitizer.
 * Built and run by tests/test_oracle_pins.py::test_oracle_under_sanitizers:
 *     gcc -O1 -g -fsanitize=address,undefined -fno-sanitize-recover=all -pthread tests/asan_driver.c -o <tmp>/asan_driver
 *     <tmp>/asan_driver <raw file> <block_size>
 * Includes the oracle's translation unit as is (test infrastructure: only tests/ may do that) and walks every entry
 * point on the given bytes: encode (three parameter sets), validate, sequential and block-parallel decode, the ASAP
 * wave simulation; exits 0 only if every decode reproduces the input.  Any out-of-bounds access, misaligned or
 * overflowing arithmetic aborts the process with a sanitizer report. */
#include "../oracle/aceapex_oracle.c"
#include <stdio.h>

int main(int argc, char** argv) {
    if (argc < 3) return 2;
    FILE* f = fopen(argv[1], "rb");
    if (!f) return 2;
    fseek(f, 0, SEEK_END); long n = ftell(f); fseek(f, 0, SEEK_SET);
    uint8_t* raw = malloc(n ? n : 1);
    if (fread(raw, 1, n, f) != (size_t)n) return 2;
    fclose(f);
    const uint32_t bs = (uint32_t)strtoul(argv[2], NULL, 10);
    const orc_enc_params sets[3] = {
        { bs, 4, 32, 0, 1, 0, 0, 0 },            /* BASELINE config 0: MIN 4, flatten on, D unlimited */
        { bs, 4, 32, 0, 0, 0, 0, 0 },            /* flatten off: deep chains */
        { bs, 4, 8, 0, 1, 2, 1, 0 },             /* depth limit 2, prefer-shallow tie break */
    };
    for (int s = 0; s < 3; ++s) {
        uint8_t* comp = NULL; uint64_t cn = 0;
        int rc = orc_encode(raw, (uint64_t)n, &sets[s], &comp, &cn);
        if (rc) { fprintf(stderr, "encode %d: %d\n", s, rc); return 1; }
        orc_report R;
        rc = orc_validate(comp, cn, &R);
        if (rc) { fprintf(stderr, "validate %d: %d\n", s, rc); return 1; }
        uint8_t* out = calloc(n ? n : 1, 1);
        if (orc_decode_seq(comp, cn, out, (uint64_t)n) || memcmp(out, raw, n)) { fprintf(stderr, "decode_seq %d\n", s); return 1; }
        memset(out, 0, n);
        if (orc_decode_mt(comp, cn, out, (uint64_t)n, 3) || memcmp(out, raw, n)) { fprintf(stderr, "decode_mt %d\n", s); return 1; }
        memset(out, 0, n);
        if (orc_asap(comp, cn, out, (uint64_t)n) < 0 || memcmp(out, raw, n)) { fprintf(stderr, "asap %d\n", s); return 1; }
        /* truncated and corrupted copies must be rejected, not read past */
        if (cn > 200) {
            uint8_t* cut = malloc(cn - 100); memcpy(cut, comp, cn - 100);
            (void)orc_validate(cut, cn - 100, &R); (void)orc_decode_seq(cut, cn - 100, out, (uint64_t)n);
            free(cut);
        }
        printf("set %d: %llu -> %llu bytes, max_depth %u, ok\n", s, (unsigned long long)n, (unsigned long long)cn, R.max_depth);
        free(out); orc_free(comp);
    }
    free(raw);
    return 0;
}
