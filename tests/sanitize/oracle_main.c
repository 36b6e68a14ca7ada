/* oracle_main.c -- TEST-ONLY driver: oracle/reshard_oracle.c compiled with -fsanitize=address,undefined and run on
 * even, uneven, empty-shard and 8-D layouts at 1, 2 and 16 bytes per element.  The check it makes on the way is an
 * invariant of the task definition: resharding A -> B -> A gives back every source shard's box.
 * tests/test_sanitizers.py builds and runs it; any sanitizer report fails the test. */
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "../../oracle/reshard_oracle.c"

static int roundtrip(const int64_t *shape, int ndim, int e, const int32_t *ma, int na, const char *sa,
                     const int32_t *mb, int nb, const char *sb) {
    int64_t la[8], lb[8], n = 1, ea = 1, eb = 1;
    int64_t da = oracle_num_devices(ma, na), db = oracle_num_devices(mb, nb);
    if (oracle_local_shape(shape, ndim, ma, na, sa, la) || oracle_local_shape(shape, ndim, mb, nb, sb, lb)) return 1;
    for (int i = 0; i < ndim; i++) { n *= shape[i]; ea *= la[i]; eb *= lb[i]; }
    unsigned char *D = malloc((size_t)(n * e));
    for (int64_t i = 0; i < n * e; i++) D[i] = (unsigned char)(i * 131u + 7u);
    void **A = malloc(sizeof(void *) * (size_t)da), **B = malloc(sizeof(void *) * (size_t)db), **A2 = malloc(sizeof(void *) * (size_t)da);
    for (int64_t r = 0; r < da; r++) {
        A[r] = calloc((size_t)(ea * e) + 1, 1); A2[r] = calloc((size_t)(ea * e) + 1, 1);
        if (oracle_shard_from_global(shape, ndim, e, ma, na, sa, r, D, A[r])) return 1;
    }
    for (int64_t q = 0; q < db; q++) B[q] = calloc((size_t)(eb * e) + 1, 1);
    int bad = reshard_oracle(shape, ndim, e, ma, na, sa, mb, nb, sb, (const void *const *)A, B, 2);
    bad |= reshard_oracle(shape, ndim, e, mb, nb, sb, ma, na, sa, (const void *const *)B, A2, 1);
    for (int64_t r = 0; r < da && !bad; r++) bad = memcmp(A[r], A2[r], (size_t)(ea * e)) != 0;   /* padding stays zero on both */
    for (int64_t r = 0; r < da; r++) { free(A[r]); free(A2[r]); }
    for (int64_t q = 0; q < db; q++) free(B[q]);
    free(A); free(A2); free(B); free(D);
    if (bad) printf("roundtrip %s -> %s failed\n", sa, sb);
    return bad;
}

int main(void) {
    int bad = 0;
    const int32_t m24[2] = {2, 4}, m42[2] = {4, 2}, m34[2] = {3, 4}, m23[2] = {2, 3}, m32[2] = {3, 2}, m4[1] = {4}, m3[1] = {3}, m2222[4] = {2, 2, 2, 2};
    const int64_t s1[2] = {8, 16}, s3[3] = {8, 16, 12}, s6[3] = {9, 10, 4}, su[3] = {7, 5, 3}, se[1] = {10}, s8[8] = {2, 3, 2, 2, 4, 2, 2, 6};
    for (int e = 1; e <= 16; e *= (e == 2 ? 8 : 2)) {
        bad += roundtrip(s1, 2, e, m24, 2, "S0,R", m24, 2, "R,S0");
        bad += roundtrip(s3, 3, e, m24, 2, "S0,S1,R", m42, 2, "S1,R,S0");
        bad += roundtrip(s6, 3, e, m24, 2, "S0,R,R", m34, 2, "S0,R,R");
        bad += roundtrip(su, 3, e, m23, 2, "S1,R,S0", m32, 2, "R,S0,S1");
        bad += roundtrip(se, 1, e, m3, 1, "S0", m4, 1, "S0");
        bad += roundtrip(s8, 8, e, m2222, 4, "S0,R,S1,R,S2,R,R,S3", m2222, 4, "R,S3,R,S2,R,S1,S0,R");
        bad += roundtrip(s3, 3, e, m24, 2, "S01,R,R", m24, 2, "R,R,S10");
    }
    printf("oracle under sanitizers: %d failures\n", bad);
    return bad ? 1 : 0;
}
