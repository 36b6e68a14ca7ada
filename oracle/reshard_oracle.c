/*
 * oracle/reshard_oracle.c -- CPU ORACLE for cross-mesh resharding (arXiv 2211.05322).
 *
 * THIS FILE IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow, obviously
 * correct statement of what a cross-mesh resharding task computes, written from the
 * paper's definitions only.  It shares no code, header, table or helper with the CUDA
 * path under paper_2211_05322_b200/csrc/ and neither includes the other.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
 *
 * What it follows (citations are PAPER.md:<line>, section):
 *   - device mesh, row-major device ids, (2,2) = [[0,1],[2,3]]      PAPER.md:78-82  (S2.2 "Device mesh")
 *   - sharding spec X_0^{d_0}...X_{N-1}^{d_{N-1}}, X in {S,R}       PAPER.md:84     (S2.2 "Sharding spec")
 *   - data slice / replica held by each device                     PAPER.md:86     (S2.2 "Data slice")
 *   - the task: send D under X_A on Mesh_A to Mesh_B under X_B      PAPER.md:88     (S2.2 "Cross-mesh resharding")
 *
 * The result is exactly defined (a relayout), so the oracle is the definition written out:
 *
 *   for every destination device q, for every local multi-index j of q's shard:
 *       g_i        = lo_i(q) + j_i                      (global index of that element)
 *       p_i        = g_i / c^A_i, c_i = ceil(l_i / k_i)  (which source shard holds it on dim i)
 *       source dev = the device whose mesh coordinates on the axes X_A uses give p, and whose
 *                    coordinates on the axes X_A does not use are 0 (lowest-index replica)
 *       dst_q[j]   = src_dev[g - lo(src_dev)]           (copy elem_bytes bytes)
 *
 * No slices, no cutpoints, no plan, no runs, no blocking: per-element index arithmetic
 * and a byte copy.  OpenMP only splits the outermost loop; every thread writes disjoint
 * elements so the result does not depend on the thread count.
 *
 * Readings of the paper used here (DESIGN.md "Readings" R1-R5, R11, R12):
 *   R1  device id = row-major rank of the mesh coordinates (last mesh axis fastest).
 *   R2  S^{ab..}: degree = prod m[a],m[b],..; shard index is the mixed-radix number with the
 *       FIRST listed axis most significant (S^{01} on (2,4): p = c0*4 + c1, degree 8).
 *   R3  one mesh axis may shard at most one tensor dim -> OR_ESPEC otherwise.
 *   R4  a mesh axis of size 1 is legal; it shards into 1 piece (behaves as R).
 *   R5  uneven partitions ("handles tiling, padding", "pad it in case 6"):
 *       every shard has the padded extent c_i = ceil(l_i / k_i); shard p holds
 *       [min(p c_i, l_i), min((p+1) c_i, l_i)) -- the last one short, later ones possibly empty.
 *       Divisible dims (all of the paper's other cases) are the special case c_i = l_i / k_i.
 *   R11 a shard buffer is dense row-major of the PADDED local shape (c_0, ..., c_{N-1}), the same on
 *       every device; the device's box sits at its origin; padding is never read and never written.
 *   R12 replicas are assumed identical; the oracle reads the lowest-index replica.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): the Fig. 2 worked example,
 * numpy basic slicing with hand-written boxes, memcpy special cases, A->B->A identity,
 * exactly-once coverage.  Nothing here is "parity unpinned".
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>
#include <ctype.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define OR_MAX_NDIM 8
#define OR_MAX_MESH_NDIM 4

enum { OR_OK = 0, OR_EINVAL = 1, OR_ESPEC = 2, OR_EDIVIS = 3 };

typedef struct {
    int n_axes;                      /* 0 => R */
    int axes[OR_MAX_MESH_NDIM];      /* listed order, first = most significant */
} or_dimspec;

typedef struct {
    int ndim;
    int64_t shape[OR_MAX_NDIM];      /* l_i */
    int mesh_ndim;
    int64_t mesh[OR_MAX_MESH_NDIM];  /* m_a */
    or_dimspec spec[OR_MAX_NDIM];
    int64_t degree[OR_MAX_NDIM];     /* k_i */
    int64_t local[OR_MAX_NDIM];      /* c_i = ceil(l_i / k_i): padded local extent (R5) */
    int64_t n_devices;
} or_layout;

/* Spec text: one entry per tensor dim, 'R' or 'S' followed by one or more mesh-axis digits.
 * Commas, spaces, parentheses, '^', '{', '}' and '_' between entries are ignored, so
 * "S0,R,S1", "(S01, R, R)", "RRR", "RS^{01}R" all parse.  PAPER.md:84. */
static int or_parse_spec(const char *s, int ndim, int mesh_ndim, or_dimspec *out)
{
    int n = 0;
    int used[OR_MAX_MESH_NDIM] = {0, 0, 0, 0};
    if (!s) return OR_EINVAL;
    while (*s) {
        char c = *s;
        if (c == ',' || c == ' ' || c == '(' || c == ')' || c == '[' || c == ']' || c == '\t') { s++; continue; }
        if (c == 'R' || c == 'r') {
            if (n >= ndim) return OR_ESPEC;
            out[n].n_axes = 0;
            n++; s++;
            continue;
        }
        if (c == 'S' || c == 's') {
            int na = 0;
            if (n >= ndim) return OR_ESPEC;
            s++;
            while (*s == '^' || *s == '{' || *s == '_' || *s == ' ') s++;
            while (isdigit((unsigned char)*s)) {
                int a = *s - '0';
                if (a >= mesh_ndim) return OR_ESPEC;
                if (used[a]) return OR_ESPEC;          /* R3 */
                if (na >= OR_MAX_MESH_NDIM) return OR_ESPEC;
                used[a] = 1;
                out[n].axes[na++] = a;
                s++;
            }
            while (*s == '}') s++;
            if (na == 0) return OR_ESPEC;
            out[n].n_axes = na;
            n++;
            continue;
        }
        return OR_ESPEC;
    }
    return n == ndim ? OR_OK : OR_ESPEC;
}

static int or_make_layout(const int64_t *shape, int ndim, const int32_t *mesh, int mesh_ndim,
                          const char *spec, or_layout *L)
{
    int i, a, rc;
    if (!shape || !mesh || !spec || !L) return OR_EINVAL;
    if (ndim < 1 || ndim > OR_MAX_NDIM) return OR_EINVAL;
    if (mesh_ndim < 1 || mesh_ndim > OR_MAX_MESH_NDIM) return OR_EINVAL;
    L->ndim = ndim;
    L->mesh_ndim = mesh_ndim;
    L->n_devices = 1;
    for (a = 0; a < mesh_ndim; a++) {
        if (mesh[a] < 1) return OR_EINVAL;
        L->mesh[a] = mesh[a];
        L->n_devices *= mesh[a];
    }
    for (i = 0; i < ndim; i++) {
        if (shape[i] < 1) return OR_EINVAL;
        L->shape[i] = shape[i];
    }
    rc = or_parse_spec(spec, ndim, mesh_ndim, L->spec);
    if (rc != OR_OK) return rc;
    for (i = 0; i < ndim; i++) {
        int64_t k = 1;
        for (a = 0; a < L->spec[i].n_axes; a++) k *= L->mesh[L->spec[i].axes[a]];
        L->degree[i] = k;
        L->local[i] = (L->shape[i] + k - 1) / k;          /* R5: ceil */
    }
    return OR_OK;
}

/* device id -> mesh coordinates, row-major ((2,2) mesh is [[0,1],[2,3]]). */
static void or_device_coords(const or_layout *L, int64_t r, int64_t *c)
{
    int a;
    for (a = L->mesh_ndim - 1; a >= 0; a--) {
        c[a] = r % L->mesh[a];
        r /= L->mesh[a];
    }
}

/* shard index of device r on tensor dim i (R2: first listed axis most significant). */
static int64_t or_shard_index(const or_layout *L, const int64_t *c, int i)
{
    int64_t p = 0;
    int a;
    for (a = 0; a < L->spec[i].n_axes; a++) {
        int ax = L->spec[i].axes[a];
        p = p * L->mesh[ax] + c[ax];
    }
    return p;
}

/* lowest-index device whose shard indices are p[0..ndim): coordinates on unused axes are 0. */
static int64_t or_owner_device(const or_layout *L, const int64_t *p)
{
    int64_t c[OR_MAX_MESH_NDIM] = {0, 0, 0, 0};
    int64_t r = 0;
    int i, a;
    for (i = 0; i < L->ndim; i++) {
        int64_t rem = p[i];
        for (a = L->spec[i].n_axes - 1; a >= 0; a--) {
            int ax = L->spec[i].axes[a];
            c[ax] = rem % L->mesh[ax];
            rem /= L->mesh[ax];
        }
    }
    for (a = 0; a < L->mesh_ndim; a++) r = r * L->mesh[a] + c[a];
    return r;
}

/* ---------------------------------------------------------------- exported queries */

int64_t oracle_num_devices(const int32_t *mesh, int mesh_ndim)
{
    int64_t n = 1;
    int a;
    if (!mesh || mesh_ndim < 1 || mesh_ndim > OR_MAX_MESH_NDIM) return -1;
    for (a = 0; a < mesh_ndim; a++) n *= mesh[a];
    return n;
}

/* (padded) local shard shape c_i = ceil(l_i / k_i) (R5). */
int oracle_local_shape(const int64_t *shape, int ndim, const int32_t *mesh, int mesh_ndim,
                       const char *spec, int64_t *local_out)
{
    or_layout L;
    int i, rc = or_make_layout(shape, ndim, mesh, mesh_ndim, spec, &L);
    if (rc != OR_OK) return rc;
    for (i = 0; i < ndim; i++) local_out[i] = L.local[i];
    return OR_OK;
}

/* the box [lo, hi) of D that device r holds. */
int oracle_device_box(const int64_t *shape, int ndim, const int32_t *mesh, int mesh_ndim,
                      const char *spec, int64_t r, int64_t *lo, int64_t *hi)
{
    or_layout L;
    int64_t c[OR_MAX_MESH_NDIM];
    int i, rc = or_make_layout(shape, ndim, mesh, mesh_ndim, spec, &L);
    if (rc != OR_OK) return rc;
    if (r < 0 || r >= L.n_devices) return OR_EINVAL;
    or_device_coords(&L, r, c);
    for (i = 0; i < ndim; i++) {
        int64_t p = or_shard_index(&L, c, i);
        lo[i] = p * L.local[i];
        hi[i] = lo[i] + L.local[i];
        if (lo[i] > L.shape[i]) lo[i] = L.shape[i];        /* R5: clipped to the tensor */
        if (hi[i] > L.shape[i]) hi[i] = L.shape[i];
    }
    return OR_OK;
}

/* Layout definition: shard_r[j] = D[lo(r) + j] for every j with lo(r) + j inside D, dense row-major
 * of the padded local shape (R5, R11); padding elements of shard_out are left as
 * the caller filled them.  D is the whole tensor, dense row-major, on the host. */
int oracle_shard_from_global(const int64_t *shape, int ndim, int elem_bytes,
                             const int32_t *mesh, int mesh_ndim, const char *spec,
                             int64_t r, const void *D, void *shard_out)
{
    or_layout L;
    int64_t c[OR_MAX_MESH_NDIM], lo[OR_MAX_NDIM], n_local = 1, j;
    int i, rc = or_make_layout(shape, ndim, mesh, mesh_ndim, spec, &L);
    if (rc != OR_OK) return rc;
    if (elem_bytes < 1 || !D || !shard_out) return OR_EINVAL;
    if (r < 0 || r >= L.n_devices) return OR_EINVAL;
    or_device_coords(&L, r, c);
    for (i = 0; i < ndim; i++) {
        lo[i] = or_shard_index(&L, c, i) * L.local[i];
        n_local *= L.local[i];
    }
    for (j = 0; j < n_local; j++) {
        int64_t rem = j, g = 0, ji[OR_MAX_NDIM];
        int pad = 0;
        for (i = ndim - 1; i >= 0; i--) { ji[i] = rem % L.local[i]; rem /= L.local[i]; }
        for (i = 0; i < ndim; i++) {
            if (lo[i] + ji[i] >= L.shape[i]) pad = 1;
            g = g * L.shape[i] + (lo[i] + ji[i]);
        }
        if (pad) continue;
        memcpy((char *)shard_out + j * elem_bytes, (const char *)D + g * elem_bytes, (size_t)elem_bytes);
    }
    return OR_OK;
}

/* where one destination element comes from: (q, local linear index j in the padded shard) ->
 * (source device, source local linear index, global linear index); source device -1 if (q, j) is
 * padding.  Used for sampled checks at sizes where running the whole oracle would take too long. */
static void or_element_source(const or_layout *A, const or_layout *B, const int64_t *lo_q,
                              int64_t j, int64_t *src_dev, int64_t *src_lin, int64_t *g_lin)
{
    int64_t ji[OR_MAX_NDIM], p[OR_MAX_NDIM], rem = j, s = 0, g = 0;
    int i;
    for (i = B->ndim - 1; i >= 0; i--) { ji[i] = rem % B->local[i]; rem /= B->local[i]; }
    for (i = 0; i < B->ndim; i++) {
        int64_t gi = lo_q[i] + ji[i];
        if (gi >= B->shape[i]) { *src_dev = -1; *src_lin = -1; if (g_lin) *g_lin = -1; return; }   /* padding */
        p[i] = gi / A->local[i];
        s = s * A->local[i] + (gi - p[i] * A->local[i]);
        g = g * A->shape[i] + gi;
    }
    *src_dev = or_owner_device(A, p);
    *src_lin = s;
    if (g_lin) *g_lin = g;
}

int oracle_element_source(const int64_t *shape, int ndim,
                          const int32_t *src_mesh, int src_mesh_ndim, const char *src_spec,
                          const int32_t *dst_mesh, int dst_mesh_ndim, const char *dst_spec,
                          int64_t q, int64_t j, int64_t *src_dev, int64_t *src_lin, int64_t *g_lin)
{
    or_layout A, B;
    int64_t c[OR_MAX_MESH_NDIM], lo[OR_MAX_NDIM], n_local = 1;
    int i, rc;
    rc = or_make_layout(shape, ndim, src_mesh, src_mesh_ndim, src_spec, &A);
    if (rc != OR_OK) return rc;
    rc = or_make_layout(shape, ndim, dst_mesh, dst_mesh_ndim, dst_spec, &B);
    if (rc != OR_OK) return rc;
    if (q < 0 || q >= B.n_devices) return OR_EINVAL;
    or_device_coords(&B, q, c);
    for (i = 0; i < ndim; i++) { lo[i] = or_shard_index(&B, c, i) * B.local[i]; n_local *= B.local[i]; }
    if (j < 0 || j >= n_local) return OR_EINVAL;
    or_element_source(&A, &B, lo, j, src_dev, src_lin, g_lin);
    return OR_OK;
}

/* one destination device q: fill dst_shard_q from the source shards. */
static void or_fill_device(const or_layout *A, const or_layout *B, int elem_bytes, int64_t q,
                           const void *const *src_shards, void *dst_shard_q, int n_threads)
{
    int64_t c[OR_MAX_MESH_NDIM], lo[OR_MAX_NDIM], inner = 1, j0;
    int i;
    or_device_coords(B, q, c);
    for (i = 0; i < B->ndim; i++) lo[i] = or_shard_index(B, c, i) * B->local[i];
    for (i = 1; i < B->ndim; i++) inner *= B->local[i];
    (void)n_threads;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(n_threads > 0 ? n_threads : 1)
#endif
    for (j0 = 0; j0 < B->local[0]; j0++) {
        int64_t t;
        for (t = 0; t < inner; t++) {
            int64_t j = j0 * inner + t, dev, s;
            or_element_source(A, B, lo, j, &dev, &s, NULL);
            if (dev < 0) continue;                         /* padding of the destination shard: untouched */
            memcpy((char *)dst_shard_q + j * elem_bytes,
                   (const char *)src_shards[dev] + s * elem_bytes, (size_t)elem_bytes);
        }
    }
}

int reshard_oracle_device(const int64_t *shape, int ndim, int elem_bytes,
                          const int32_t *src_mesh, int src_mesh_ndim, const char *src_spec,
                          const int32_t *dst_mesh, int dst_mesh_ndim, const char *dst_spec,
                          const void *const *src_shards, int64_t q, void *dst_shard_q, int n_threads)
{
    or_layout A, B;
    int rc;
    if (elem_bytes < 1 || !src_shards || !dst_shard_q) return OR_EINVAL;
    rc = or_make_layout(shape, ndim, src_mesh, src_mesh_ndim, src_spec, &A);
    if (rc != OR_OK) return rc;
    rc = or_make_layout(shape, ndim, dst_mesh, dst_mesh_ndim, dst_spec, &B);
    if (rc != OR_OK) return rc;
    if (q < 0 || q >= B.n_devices) return OR_EINVAL;
    or_fill_device(&A, &B, elem_bytes, q, src_shards, dst_shard_q, n_threads);
    return OR_OK;
}

/* the whole task: every destination device.  src_shards[r] / dst_shards[q] are
 * host pointers indexed by row-major device id; only the lowest-index replica of each source
 * tile is dereferenced, so a harness may alias replicas to one buffer. */
int reshard_oracle(const int64_t *shape, int ndim, int elem_bytes,
                   const int32_t *src_mesh, int src_mesh_ndim, const char *src_spec,
                   const int32_t *dst_mesh, int dst_mesh_ndim, const char *dst_spec,
                   const void *const *src_shards, void *const *dst_shards, int n_threads)
{
    or_layout A, B;
    int64_t q;
    int rc;
    if (elem_bytes < 1 || !src_shards || !dst_shards) return OR_EINVAL;
    rc = or_make_layout(shape, ndim, src_mesh, src_mesh_ndim, src_spec, &A);
    if (rc != OR_OK) return rc;
    rc = or_make_layout(shape, ndim, dst_mesh, dst_mesh_ndim, dst_spec, &B);
    if (rc != OR_OK) return rc;
    for (q = 0; q < B.n_devices; q++)
        or_fill_device(&A, &B, elem_bytes, q, src_shards, dst_shards[q], n_threads);
    return OR_OK;
}

/* threads OpenMP will really use for a request of n (sched affinity is honoured by libgomp). */
int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_num_procs();
#else
    return 1;
#endif
}
