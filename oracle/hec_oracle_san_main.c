/*
 * TEST INFRASTRUCTURE ONLY -- command-line driver of oracle/hec_oracle.c for the sanitizer build
 * (tests/test_oracle_sanitizers.py: gcc -fsanitize=address,undefined).
 *
 *   hec_oracle_san p r g k_hi in.bin out.bin
 *
 * in.bin  : n rows of 2g+3 uint16 coefficients (row-major, c_0 first)
 * out.bin : n rows of k_hi uint32 counts N_1..N_k_hi, then n rows of k_hi uint32 root counts r0_1..r0_k_hi,
 *           then n bytes squarefree flag
 * Also exercises the modulus entry points (smallest irreducible / primitive, multiplication) once, so that
 * their stack arrays run under the sanitizers too.  No arithmetic of its own.
 */
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

int orc_smallest_irreducible(uint32_t p, uint32_t n, uint32_t *out);
int orc_smallest_primitive(uint32_t p, uint32_t n, uint32_t *out);
int orc_is_primitive(uint32_t p, uint32_t n, const uint32_t *mod);
long long orc_mul_encoded(uint32_t p, uint32_t n, const uint32_t *mod, uint64_t a, uint64_t b);
int orc_count_range(uint32_t p, uint32_t r, uint32_t g, const uint16_t *coeffs, size_t n, uint32_t k_lo, uint32_t k_hi,
                    uint32_t width, uint32_t *out_counts, uint8_t *out_squarefree, int nthreads, int *threads_used);
int orc_roots_range(uint32_t p, uint32_t r, uint32_t g, const uint16_t *coeffs, size_t n, uint32_t k_lo, uint32_t k_hi,
                    uint32_t width, uint32_t *out_roots, int nthreads);

int main(int argc, char **argv) {
    if (argc != 7) { fprintf(stderr, "usage: %s p r g k_hi in.bin out.bin\n", argv[0]); return 2; }
    const uint32_t p = (uint32_t)atoi(argv[1]), r = (uint32_t)atoi(argv[2]), g = (uint32_t)atoi(argv[3]), k_hi = (uint32_t)atoi(argv[4]);
    const uint32_t ncoef = 2 * g + 3;
    FILE *fi = fopen(argv[5], "rb");
    if (!fi) { perror("in"); return 2; }
    fseek(fi, 0, SEEK_END);
    const long bytes = ftell(fi);
    fseek(fi, 0, SEEK_SET);
    const size_t n = (size_t)bytes / (2 * ncoef);
    uint16_t *rows = malloc(n * ncoef * sizeof *rows);
    uint32_t *cnt = calloc(n * k_hi, sizeof *cnt), *r0 = calloc(n * k_hi, sizeof *r0);
    uint8_t *sf = calloc(n, 1);
    if (!rows || !cnt || !r0 || !sf || fread(rows, 2 * ncoef, n, fi) != n) { fprintf(stderr, "read failed\n"); return 2; }
    fclose(fi);

    uint32_t mod[16];
    for (uint32_t deg = 1; deg <= r * k_hi; deg++) {
        if (orc_smallest_irreducible(p, deg, mod)) return 3;
        if (orc_smallest_primitive(p, deg, mod)) return 3;
        if (orc_is_primitive(p, deg, mod) != 1) return 3;
        if (orc_mul_encoded(p, deg, mod, 1, 1) != 1) return 3;
    }
    int used = 0;
    int rc = orc_count_range(p, r, g, rows, n, 1, k_hi, k_hi, cnt, sf, 0, &used);
    if (rc) { fprintf(stderr, "orc_count_range: %d\n", rc); return 4; }
    rc = orc_roots_range(p, r, g, rows, n, 1, k_hi, k_hi, r0, 0);
    if (rc) { fprintf(stderr, "orc_roots_range: %d\n", rc); return 4; }

    FILE *fo = fopen(argv[6], "wb");
    if (!fo) { perror("out"); return 2; }
    fwrite(cnt, sizeof *cnt, n * k_hi, fo);
    fwrite(r0, sizeof *r0, n * k_hi, fo);
    fwrite(sf, 1, n, fo);
    fclose(fo);
    free(rows); free(cnt); free(r0); free(sf);
    return 0;
}
