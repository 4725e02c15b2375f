/*
 * oracle/pic_ref.c -- plain, slow, obviously-correct CPU statement of the particle
 * hot path of PIC_ENGINE (arXiv 1603.02886): sort by cell key, B-spline charge
 * deposit, field gather + accel + push.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference leg may load it.  It shares no
 * code, header, table or constant with paper_1603_02886_b200/ (the CUDA path).
 *
 * Arithmetic: double throughout, on the stored fp32/fp64 inputs converted exactly
 * to double; x and v are rounded ONCE to the storage dtype on output; rho stays
 * double.  The single exception is t = x/h, which is an IEEE division in the
 * STORAGE precision (reading R13) so that the integer cell index is
 * decided in the same precision on both sides.  Single thread, particle order,
 * stencil loops z-outer / y / x-inner.  No blocking, fusion or reordering.
 *
 * A second, TIMED-ONLY build (oracle.build_openmp(): the same file with -fopenmp,
 * libpicref_omp.so) spreads the particle loops of the key pass, the attribute move,
 * the deposit (one private grid per thread, added up node by node at the end) and the push over
 * the host cores: it mirrors the paper's own CPU reference, OpenMP on 8 cores
 * (PAPER.md:388), for bench.py's cpu_baseline.  Everything between `#ifdef _OPENMP`
 * belongs to that build; the parity tests load the plain build only, whose
 * arithmetic and order are as stated above.
 *
 * Every function cites the passage of /root/reference/PAPER.md it follows
 * (PAPER.md:NNN = line NNN, with section).  Readings R1..R20 of silent or garbled
 * passages are listed in DESIGN.md.
 *
 * Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`): B-spline closed forms,
 * partition of unity and moments; the paper's 8 trilinear products;
 * exact charge conservation; one-particle closed-form deposits; all-pairs brute
 * force (the paper's threads-on-grid definition); numpy stable
 * argsort; gather/deposit adjointness; analytic push under one Fourier mode.
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>                                         /* timed OpenMP build only, see the header */
#endif

typedef struct {
    int32_t dim;      /* 2 or 3 */
    int32_t n[3];     /* cells = nodes per dimension (periodic); n[2] = 1 if dim == 2 */
    double  h[3];     /* spacing; node j sits at j*h; box length L = n*h */
    int32_t order;    /* B-spline degree p: 1, 2, 3 */
    int32_t dtype;    /* storage dtype of particles and E: 0 = fp32, 1 = fp64 */
} pic_ref_grid;

enum { REF_OK = 0, REF_BAD_ARG = -1 };

static int grid_ok(const pic_ref_grid *g)
{
    if (!g || (g->dim != 2 && g->dim != 3)) return 0;
    if (g->order < 1 || g->order > 3) return 0;
    if (g->dtype != 0 && g->dtype != 1) return 0;
    for (int c = 0; c < g->dim; ++c)
        if (g->n[c] < g->order + 1 || !(g->h[c] > 0.0)) return 0;
    return 1;
}

static int64_t grid_cells(const pic_ref_grid *g)
{
    int64_t C = 1;
    for (int c = 0; c < g->dim; ++c) C *= g->n[c];
    return C;
}

static double load_real(const pic_ref_grid *g, const void *a, int64_t i)
{
    return g->dtype ? ((const double *)a)[i] : (double)((const float *)a)[i];
}

static void store_real(const pic_ref_grid *g, void *a, int64_t i, double v)
{
    if (g->dtype) ((double *)a)[i] = v;
    else          ((float *)a)[i] = (float)v;
}

/* t = x/h evaluated by IEEE division in the storage precision (reading R13);
 * the paper works in grid units, ix=(int)x (App. B). */
static double grid_coord(const pic_ref_grid *g, int c, const void *x, int64_t i)
{
    if (g->dtype) return ((const double *)x)[i] / g->h[c];
    volatile float q = ((const float *)x)[i] / (float)g->h[c];
    return (double)q;
}

/* Clamped cell index, PAPER.md:493-497 (App. B: "if (ix<0) ix=0; if (ix>nx-1) ix=nx-1"). */
static int32_t cell_index(const pic_ref_grid *g, int c, double t)
{
    double f = floor(t);
    if (f < 0.0) return 0;
    if (f > (double)(g->n[c] - 1)) return g->n[c] - 1;
    return (int32_t)f;
}

/* ---------------------------------------------------------------------------
 * O1. Centred cardinal B-spline of degree p, closed piecewise form.
 * p = 1 is PAPER.md:455-461 verbatim: MIN(1-w,1+w) for ABS(w) <= 1 (App. B, Fortran).
 * p = 2, 3: the "higher order B-splines" the paper names; reading R1.
 * ------------------------------------------------------------------------- */
double pic_ref_bspline(int p, double t)
{
    double a = fabs(t);
    switch (p) {
    case 1:
        return a <= 1.0 ? 1.0 - a : 0.0;
    case 2:
        if (a <= 0.5) return 0.75 - a * a;
        if (a <= 1.5) return 0.5 * (1.5 - a) * (1.5 - a);
        return 0.0;
    case 3:
        if (a <= 1.0) return 2.0 / 3.0 - a * a + 0.5 * a * a * a;
        if (a <= 2.0) return (2.0 - a) * (2.0 - a) * (2.0 - a) / 6.0;
        return 0.0;
    default:
        return 0.0;
    }
}

/* ---------------------------------------------------------------------------
 * O1. Stencil form in one dimension: with t = x/h, i0 = clamped floor(t) (the
 * same index as the key), xi = t - i0, the p+1 nodes carrying weight and their
 * weights.  p = 1 gives (1-xi, xi), i.e. the factors of the paper's 8 products
 * (PAPER.md:509-519).  Node indices are folded mod n (periodic).
 * Returns p+1.
 * ------------------------------------------------------------------------- */
static int stencil_1d(const pic_ref_grid *g, int c, double t, int32_t idx[4], double wt[4])
{
    int32_t n = g->n[c];
    int32_t i0 = cell_index(g, c, t);
    double xi = t - (double)i0;
    int32_t first;
    int m = g->order + 1;
    if (g->order == 1) {
        first = i0;
        wt[0] = 1.0 - xi;
        wt[1] = xi;
    } else if (g->order == 2) {
        int32_t j = i0 + (xi >= 0.5 ? 1 : 0);         /* nearest node */
        double d = xi - (double)(j - i0);             /* in [-1/2, 1/2] */
        first = j - 1;
        wt[0] = 0.5 * (0.5 - d) * (0.5 - d);
        wt[1] = 0.75 - d * d;
        wt[2] = 0.5 * (0.5 + d) * (0.5 + d);
    } else {
        double x2 = xi * xi, x3 = x2 * xi, om = 1.0 - xi;
        first = i0 - 1;
        wt[0] = om * om * om / 6.0;
        wt[1] = (3.0 * x3 - 6.0 * x2 + 4.0) / 6.0;
        wt[2] = (-3.0 * x3 + 3.0 * x2 + 3.0 * xi + 1.0) / 6.0;
        wt[3] = x3 / 6.0;
    }
    for (int a = 0; a < m; ++a) {
        int32_t j = (first + a) % n;
        idx[a] = j < 0 ? j + n : j;
    }
    return m;
}

/* exposed for the pins: stencil of particle i in dimension c */
int pic_ref_stencil_1d(const pic_ref_grid *g, int c, const void *x, int64_t i,
                       int32_t *idx, double *wt)
{
    if (!grid_ok(g) || c < 0 || c >= g->dim) return REF_BAD_ARG;
    return stencil_1d(g, c, grid_coord(g, c, x, i), idx, wt);
}

/* ---------------------------------------------------------------------------
 * a1. Cell key: the particle's target bucket (section 3.2), one cell
 * per bucket, bins ordered x fastest.
 * ------------------------------------------------------------------------- */
static int32_t cell_key(const pic_ref_grid *g, const void *const x[3], int64_t i)
{
    int64_t key = 0, stride = 1;
    for (int c = 0; c < g->dim; ++c) {
        key += stride * cell_index(g, c, grid_coord(g, c, x[c], i));
        stride *= g->n[c];
    }
    return (int32_t)key;
}

int pic_ref_keys(const pic_ref_grid *g, int64_t n, const void *const x[3], int32_t *key)
{
    if (!grid_ok(g) || n < 0) return REF_BAD_ARG;
    for (int64_t i = 0; i < n; ++i) key[i] = cell_key(g, x, i);
    return REF_OK;
}

/* ---------------------------------------------------------------------------
 * O2 / a2-a4. Counting sort by cell key: histogram, exclusive prefix sum, scatter
 * (section 3.2, Sintorn-Assarsson bucket sort; Alg. 2
 * lines 1-5).  The paper's atomic counters leave the order inside a bucket
 * arbitrary; here particles are visited in ascending source index so the sort is
 * STABLE and perm is unique (reading R7).  Out of place; the
 * caller ping-pongs instead of copying back.  perm[j] = source index of the
 * particle now at j (reading R9).
 * ------------------------------------------------------------------------- */
int pic_ref_sort(const pic_ref_grid *g, int64_t n,
                 const void *const xin[3], const void *const vin[3], const void *win,
                 void *const xout[3], void *const vout[3], void *wout,
                 int32_t *perm, int32_t *cell_offsets)
{
    if (!grid_ok(g) || n < 0 || n > 2147483647LL) return REF_BAD_ARG;
    int64_t C = grid_cells(g);
    int32_t *key = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    int32_t *cursor = (int32_t *)malloc(sizeof(int32_t) * (size_t)(C + 1));
    if (!key || !cursor) { free(key); free(cursor); return REF_BAD_ARG; }

    for (int64_t k = 0; k <= C; ++k) cell_offsets[k] = 0;
#ifdef _OPENMP                                           /* timed OpenMP build only, see the header */
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        key[i] = cell_key(g, xin, i);
#pragma omp atomic
        cell_offsets[key[i] + 1] += 1;
    }
#else
    for (int64_t i = 0; i < n; ++i) {                    /* histogram */
        key[i] = cell_key(g, xin, i);
        cell_offsets[key[i] + 1] += 1;
    }
#endif
    for (int64_t k = 0; k < C; ++k)                      /* prefix sum */
        cell_offsets[k + 1] += cell_offsets[k];
    for (int64_t k = 0; k < C; ++k) cursor[k] = cell_offsets[k];
    for (int64_t i = 0; i < n; ++i)                      /* stable scatter */
        perm[cursor[key[i]]++] = (int32_t)i;

    size_t s = g->dtype ? 8 : 4;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int64_t j = 0; j < n; ++j) {                    /* move the attributes bit for bit */
        int64_t i = perm[j];
        for (int c = 0; c < g->dim; ++c) {
            memcpy((char *)xout[c] + s * j, (const char *)xin[c] + s * i, s);
            memcpy((char *)vout[c] + s * j, (const char *)vin[c] + s * i, s);
        }
        memcpy((char *)wout + s * j, (const char *)win + s * i, s);
    }
    free(key);
    free(cursor);
    return REF_OK;
}

/* ---------------------------------------------------------------------------
 * NEXT-2. Buckets of several cells (section 3.2: "a bucket ... one or more grid
 * cells"; App. B: "ibin = bin % nsplitx; jbin = bin / nsplitx", bins ordered x
 * fastest; the bucket-count sweep of PAPER.md:336-350 Fig. 9 and 396-402 Fig. 14).
 * A bucket is a box of bucket[c] cells per dimension (the last one of a dimension is smaller
 * when bucket[c] does not divide n[c]); there are nb[c] = ceil(n[c] / bucket[c]) per dimension.
 *   key_i = b_x + nb_x (b_y + nb_y b_z),  b_c = floor(cell_c / bucket[c]),
 * cell_c the clamped cell index of a1.  The sort is the same stable counting sort with this
 * key: particles of one bucket become contiguous and keep their source order inside it (the
 * paper leaves that order arbitrary).  bucket = (1,1,1) is pic_ref_sort.
 * ------------------------------------------------------------------------- */
static int bucket_ok(const pic_ref_grid *g, const int32_t bucket[3])
{
    for (int c = 0; c < g->dim; ++c)
        if (bucket[c] < 1 || bucket[c] > g->n[c]) return 0;
    return 1;
}

int64_t pic_ref_bucket_count(const pic_ref_grid *g, const int32_t bucket[3])
{
    if (!grid_ok(g) || !bucket_ok(g, bucket)) return -1;
    int64_t B = 1;
    for (int c = 0; c < g->dim; ++c) B *= (g->n[c] + bucket[c] - 1) / bucket[c];
    return B;
}

static int32_t bucket_key(const pic_ref_grid *g, const int32_t bucket[3], const void *const x[3], int64_t i)
{
    int64_t key = 0, stride = 1;
    for (int c = 0; c < g->dim; ++c) {
        int32_t cell = cell_index(g, c, grid_coord(g, c, x[c], i));
        key += stride * (cell / bucket[c]);
        stride *= (g->n[c] + bucket[c] - 1) / bucket[c];
    }
    return (int32_t)key;
}

int pic_ref_bucket_keys(const pic_ref_grid *g, const int32_t bucket[3], int64_t n, const void *const x[3], int32_t *key)
{
    if (!grid_ok(g) || !bucket_ok(g, bucket) || n < 0) return REF_BAD_ARG;
    for (int64_t i = 0; i < n; ++i) key[i] = bucket_key(g, bucket, x, i);
    return REF_OK;
}

int pic_ref_sort_buckets(const pic_ref_grid *g, const int32_t bucket[3], int64_t n,
                         const void *const xin[3], const void *const vin[3], const void *win,
                         void *const xout[3], void *const vout[3], void *wout,
                         int32_t *perm, int32_t *bucket_offsets)
{
    if (!grid_ok(g) || !bucket_ok(g, bucket) || n < 0 || n > 2147483647LL) return REF_BAD_ARG;
    int64_t B = pic_ref_bucket_count(g, bucket);
    int32_t *key = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    int32_t *cursor = (int32_t *)malloc(sizeof(int32_t) * (size_t)(B + 1));
    if (!key || !cursor) { free(key); free(cursor); return REF_BAD_ARG; }
    for (int64_t k = 0; k <= B; ++k) bucket_offsets[k] = 0;
    for (int64_t i = 0; i < n; ++i) {                    /* histogram */
        key[i] = bucket_key(g, bucket, xin, i);
        bucket_offsets[key[i] + 1] += 1;
    }
    for (int64_t k = 0; k < B; ++k)                      /* prefix sum */
        bucket_offsets[k + 1] += bucket_offsets[k];
    for (int64_t k = 0; k < B; ++k) cursor[k] = bucket_offsets[k];
    for (int64_t i = 0; i < n; ++i)                      /* stable scatter */
        perm[cursor[key[i]]++] = (int32_t)i;
    size_t s = g->dtype ? 8 : 4;
    for (int64_t j = 0; j < n; ++j) {                    /* move the attributes bit for bit */
        int64_t i = perm[j];
        for (int c = 0; c < g->dim; ++c) {
            memcpy((char *)xout[c] + s * j, (const char *)xin[c] + s * i, s);
            memcpy((char *)vout[c] + s * j, (const char *)vin[c] + s * i, s);
        }
        memcpy((char *)wout + s * j, (const char *)win + s * i, s);
    }
    free(key);
    free(cursor);
    return REF_OK;
}

/* ---------------------------------------------------------------------------
 * NEXT-1. "Bucketsort for pre-ordered particles, contiguous datastructure" (Alg. 2; text
 * PAPER.md:190-196): the sort the paper prefers ("for the rest of this paper this sorting algorithm is
 * considered").  IN PLACE; only the misplaced particles move.  Steps, in the listing's order:
 *   l.1-5   bucket_sizes = histogram of the keys, bucket_offsets = prefix sum
 *   l.6-10  bucket_num[ip] = the bucket whose region [offsets[b], offsets[b+1]) holds array position ip
 *   l.13-20 a particle is misplaced if bucket_num[ip] != key(ip); counts per bucket, offsets of the buffers
 *   l.21-30 misplaced particles go to particles_buffer (grouped by TARGET bucket), their positions to holes_buffer
 *           (grouped by SOURCE bucket = region)
 *   l.31-35 the particles of the buffer are put into the holes of their target bucket
 * The paper takes buffer slots with atomic counters, so which incoming particle lands in which hole of its bucket is
 * arbitrary.  Reading (R24): slots in ascending array position on both sides -- the holes of a region in
 * ascending position, the incoming particles of a bucket in ascending source position -- which makes the result
 * unique.  Region b has as many holes as there are misplaced particles with key b (both equal bucket_sizes[b] minus
 * the particles of key b already inside the region), so hole i of the whole array (ascending) receives misplaced
 * particle i of the list sorted stably by key.  Not a stable sort: particles already in their region do not move.
 * *moved = number of misplaced particles.  bucket = (1,1,1): cells.
 * ------------------------------------------------------------------------- */
int pic_ref_sort_buckets_inplace(const pic_ref_grid *g, const int32_t bucket[3], int64_t n,
                                 void *const x[3], void *const v[3], void *w,
                                 int32_t *bucket_offsets, int64_t *moved)
{
    if (!grid_ok(g) || !bucket_ok(g, bucket) || n < 0 || n > 2147483647LL) return REF_BAD_ARG;
    int64_t B = pic_ref_bucket_count(g, bucket);
    size_t s = g->dtype ? 8 : 4;
    int A = 2 * g->dim + 1;
    int32_t *key = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    int32_t *bucket_num = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    int32_t *buffer_sizes = (int32_t *)calloc((size_t)(B + 1), sizeof(int32_t));
    int32_t *buffer_offsets = (int32_t *)calloc((size_t)(B + 1), sizeof(int32_t));
    int32_t *counter_pbuffer = (int32_t *)calloc((size_t)(B + 1), sizeof(int32_t));
    if (!key || !bucket_num || !buffer_sizes || !buffer_offsets || !counter_pbuffer) return REF_BAD_ARG;
    void *arr[7];
    for (int c = 0; c < g->dim; ++c) { arr[c] = x[c]; arr[g->dim + c] = v[c]; }
    arr[2 * g->dim] = w;

    for (int64_t k = 0; k <= B; ++k) bucket_offsets[k] = 0;                 /* l.1-5 */
    for (int64_t i = 0; i < n; ++i) {
        key[i] = bucket_key(g, bucket, (const void *const *)x, i);
        bucket_offsets[key[i] + 1] += 1;
    }
    for (int64_t k = 0; k < B; ++k) bucket_offsets[k + 1] += bucket_offsets[k];
    for (int64_t b = 0; b < B; ++b)                                          /* l.6-10 */
        for (int64_t ic = bucket_offsets[b]; ic < bucket_offsets[b + 1]; ++ic) bucket_num[ic] = (int32_t)b;
    int64_t M = 0;                                                           /* l.13-17: incoming per TARGET bucket */
    for (int64_t ip = 0; ip < n; ++ip)
        if (bucket_num[ip] != key[ip]) { buffer_sizes[key[ip]] += 1; ++M; }
    for (int64_t b = 0; b < B; ++b) buffer_offsets[b + 1] = buffer_offsets[b] + buffer_sizes[b];   /* l.18-20 */
    char *particles_buffer = (char *)malloc((size_t)(M > 0 ? M : 1) * (size_t)A * s);
    int32_t *holes_buffer = (int32_t *)malloc(sizeof(int32_t) * (size_t)(M > 0 ? M : 1));
    if (!particles_buffer || !holes_buffer) return REF_BAD_ARG;
    int64_t nholes = 0;
    for (int64_t ip = 0; ip < n; ++ip) {                                     /* l.21-30, ascending position */
        int32_t source_bucket = bucket_num[ip], target_bucket = key[ip];
        if (target_bucket != source_bucket) {
            int64_t lcpbuffer = counter_pbuffer[target_bucket]++;
            int64_t slot = lcpbuffer + buffer_offsets[target_bucket];
            for (int a = 0; a < A; ++a)
                memcpy(particles_buffer + ((size_t)slot * (size_t)A + (size_t)a) * s, (const char *)arr[a] + s * (size_t)ip, s);
            holes_buffer[nholes++] = (int32_t)ip;          /* regions are ordered by position: grouped by source bucket */
        }
    }
    for (int64_t i = 0; i < M; ++i)                                          /* l.31-35 */
        for (int a = 0; a < A; ++a)
            memcpy((char *)arr[a] + s * (size_t)holes_buffer[i], particles_buffer + ((size_t)i * (size_t)A + (size_t)a) * s, s);
    if (moved) *moved = M;
    free(key); free(bucket_num); free(buffer_sizes); free(buffer_offsets); free(counter_pbuffer);
    free(particles_buffer); free(holes_buffer);
    return REF_OK;
}

/* ---------------------------------------------------------------------------
 * O3 / a5. Charge deposit (setrho, threads-on-particles form without the threads:
 * PAPER.md:292-294 section 3.3.4; the 8 products of PAPER.md:509-519 for p = 1).
 *   rho[j] = h^-d sum_i w_i prod_c W_p(x_ic/h_c - j_c)   on the periodic grid.
 * The paper adds bare products (no w, no 1/h^d); weights and the
 * normalisation are reading R2, chosen so that sum_j rho_j h^d = sum_i w_i.
 * rho is overwritten (reading R10).  Particle order; nodes z-outer/y/x-inner.
 * ------------------------------------------------------------------------- */
static void deposit_one(const pic_ref_grid *g, const void *const x[3], const void *w, int64_t i,
                        double inv_vol, double *rho)
{
    int32_t ix[3][4];
    double wt[3][4];
    int m[3] = {1, 1, 1};
    ix[2][0] = 0; wt[2][0] = 1.0;
    for (int c = 0; c < g->dim; ++c)
        m[c] = stencil_1d(g, c, grid_coord(g, c, x[c], i), ix[c], wt[c]);
    double q = load_real(g, w, i) * inv_vol;
    for (int kz = 0; kz < m[2]; ++kz)
        for (int ky = 0; ky < m[1]; ++ky)
            for (int kx = 0; kx < m[0]; ++kx) {
                int64_t j = ix[0][kx] + (int64_t)g->n[0] * (ix[1][ky] + (int64_t)g->n[1] * ix[2][kz]);
                rho[j] += q * (wt[0][kx] * wt[1][ky] * wt[2][kz]);
            }
}

int pic_ref_deposit(const pic_ref_grid *g, int64_t n, const void *const x[3], const void *w,
                    double *rho)
{
    if (!grid_ok(g) || n < 0) return REF_BAD_ARG;
    int64_t C = grid_cells(g);
    double inv_vol = 1.0;
    for (int c = 0; c < g->dim; ++c) inv_vol /= g->h[c];
    for (int64_t k = 0; k < C; ++k) rho[k] = 0.0;

#ifdef _OPENMP
    /* Timed OpenMP build only (see the header): particles split over the threads, one private grid per
     * thread, the grids added up at the end.  The summation order differs from the plain build. */
    int max_threads = omp_get_max_threads(), bad = 0;
    double **priv = (double **)calloc((size_t)max_threads, sizeof(double *));
    if (!priv) return REF_BAD_ARG;
#pragma omp parallel
    {
        int t = omp_get_thread_num(), nt = omp_get_num_threads();
        priv[t] = (double *)calloc((size_t)C, sizeof(double));
        if (!priv[t]) {
#pragma omp atomic write
            bad = 1;
        }
#pragma omp barrier
        if (!bad) {
#pragma omp for schedule(static)
            for (int64_t i = 0; i < n; ++i) deposit_one(g, x, w, i, inv_vol, priv[t]);
            /* the grids are added up node by node, threads in ascending order: parallel over the nodes, no critical
             * section */
#pragma omp for schedule(static)
            for (int64_t k = 0; k < C; ++k) {
                double sum = 0.0;
                for (int u = 0; u < nt; ++u) sum += priv[u][k];
                rho[k] = sum;
            }
        }
    }
    for (int u = 0; u < max_threads; ++u) free(priv[u]);
    free(priv);
    if (bad) return REF_BAD_ARG;
#else
    for (int64_t i = 0; i < n; ++i) deposit_one(g, x, w, i, inv_vol, rho);
#endif
    return REF_OK;
}

/* minimum image of t modulo n (periodic distance in grid units) */
static double min_image(double t, int32_t n)
{
    return t - (double)n * floor(t / (double)n + 0.5);
}

/* ---------------------------------------------------------------------------
 * O3, second and independent formulation: ALL PAIRS (node x particle).  This is the
 * paper's collision-free "threads on splines" algorithm with a single bucket
 * (section 3.3.1; App. B Fortran PAPER.md:447-469): every node loops
 * over every particle and adds the spline value if the particle is inside its
 * support.  Uses only the closed-form W_p and the minimum image; shares nothing
 * with stencil_1d.  O(C*N): tiny inputs only.
 * ------------------------------------------------------------------------- */
int pic_ref_deposit_allpairs(const pic_ref_grid *g, int64_t n, const void *const x[3],
                             const void *w, double *rho)
{
    if (!grid_ok(g) || n < 0) return REF_BAD_ARG;
    double inv_vol = 1.0;
    for (int c = 0; c < g->dim; ++c) inv_vol /= g->h[c];
    int32_t nz = g->dim == 3 ? g->n[2] : 1;
    for (int32_t jz = 0; jz < nz; ++jz)
        for (int32_t jy = 0; jy < g->n[1]; ++jy)
            for (int32_t jx = 0; jx < g->n[0]; ++jx) {
                int32_t jj[3] = {jx, jy, jz};
                double acc = 0.0;
                for (int64_t i = 0; i < n; ++i) {
                    double prod = load_real(g, w, i);
                    for (int c = 0; c < g->dim; ++c) {
                        double t = grid_coord(g, c, x[c], i);
                        prod *= pic_ref_bspline(g->order, min_image(t - (double)jj[c], g->n[c]));
                    }
                    acc += prod;
                }
                rho[jx + (int64_t)g->n[0] * (jy + (int64_t)g->n[1] * jz)] = acc * inv_vol;
            }
    return REF_OK;
}

/* ---------------------------------------------------------------------------
 * O4 / a6 (first half). Field at the particle: "an interpolation ... to obtain the
 * fields at the particle position from the fields on the nearest grid points"
 * (section 3), with the SAME B-splines as the deposit, from
 * three separate grids Ex, Ey, Ez (section 4.2).  Full (p+1)^d stencil
 * (reading R11).   Ep[c][i] = sum_j E_c[j] prod_c' W_p(x_ic'/h_c' - j_c').
 * ------------------------------------------------------------------------- */
static void gather_one(const pic_ref_grid *g, const void *const x[3], const void *const E[3],
                       int64_t i, double Ep[3])
{
    int32_t ix[3][4];
    double wt[3][4];
    int m[3] = {1, 1, 1};
    ix[2][0] = 0; wt[2][0] = 1.0;
    for (int c = 0; c < g->dim; ++c)
        m[c] = stencil_1d(g, c, grid_coord(g, c, x[c], i), ix[c], wt[c]);
    for (int c = 0; c < g->dim; ++c) {
        double acc = 0.0;
        for (int kz = 0; kz < m[2]; ++kz)
            for (int ky = 0; ky < m[1]; ++ky)
                for (int kx = 0; kx < m[0]; ++kx) {
                    int64_t j = ix[0][kx] + (int64_t)g->n[0] * (ix[1][ky] + (int64_t)g->n[1] * ix[2][kz]);
                    acc += (wt[0][kx] * wt[1][ky] * wt[2][kz]) * load_real(g, E[c], j);
                }
        Ep[c] = acc;
    }
}

int pic_ref_gather(const pic_ref_grid *g, int64_t n, const void *const x[3],
                   const void *const E[3], double *const Ep[3])
{
    if (!grid_ok(g) || n < 0) return REF_BAD_ARG;
    for (int64_t i = 0; i < n; ++i) {
        double e[3];
        gather_one(g, x, E, i, e);
        for (int c = 0; c < g->dim; ++c) Ep[c][i] = e[c];
    }
    return REF_OK;
}

/* Brute-force gather: sum over ALL nodes of E_c[j] W_p(min-image), closed form only. */
int pic_ref_gather_allnodes(const pic_ref_grid *g, int64_t n, const void *const x[3],
                            const void *const E[3], double *const Ep[3])
{
    if (!grid_ok(g) || n < 0) return REF_BAD_ARG;
    int32_t nz = g->dim == 3 ? g->n[2] : 1;
    for (int64_t i = 0; i < n; ++i) {
        double t[3] = {0, 0, 0};
        for (int c = 0; c < g->dim; ++c) t[c] = grid_coord(g, c, x[c], i);
        for (int cc = 0; cc < g->dim; ++cc) {
            double acc = 0.0;
            for (int32_t jz = 0; jz < nz; ++jz)
                for (int32_t jy = 0; jy < g->n[1]; ++jy)
                    for (int32_t jx = 0; jx < g->n[0]; ++jx) {
                        int32_t jj[3] = {jx, jy, jz};
                        double prod = 1.0;
                        for (int c = 0; c < g->dim; ++c)
                            prod *= pic_ref_bspline(g->order, min_image(t[c] - (double)jj[c], g->n[c]));
                        acc += prod * load_real(g, E[cc], jx + (int64_t)g->n[0] * (jy + (int64_t)g->n[1] * jz));
                    }
            Ep[cc][i] = acc;
        }
    }
    return REF_OK;
}

/* ---------------------------------------------------------------------------
 * O4 / a6-a7. accel then push (section 3):
 *   iii. v(t+1) = v(t) + dt * E(t)      (times q/m, reading R3; E at x(t))
 *   iv.  x(t+1) = x(t) + dt * v(t+1)    (the NEW velocity)
 * periodic boundary conditions: x -= L*floor(x/L).  Rounded once to
 * the storage dtype; a stored value >= L or < 0 becomes 0 (0 and L are the same
 * point), so 0 <= x < L always holds in storage.  In place.
 * ------------------------------------------------------------------------- */
int pic_ref_push(const pic_ref_grid *g, int64_t n, void *const x[3], void *const v[3],
                 const void *const E[3], double dt, double qm)
{
    if (!grid_ok(g) || n < 0) return REF_BAD_ARG;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int64_t i = 0; i < n; ++i) {
        double e[3];
        gather_one(g, (const void *const *)x, E, i, e);
        for (int c = 0; c < g->dim; ++c) {
            double L = (double)g->n[c] * g->h[c];
            double vn = load_real(g, v[c], i) + qm * dt * e[c];
            double xn = load_real(g, x[c], i) + dt * vn;
            xn -= L * floor(xn / L);
            store_real(g, v[c], i, vn);
            store_real(g, x[c], i, xn);
            double xs = load_real(g, x[c], i);
            if (xs >= L || xs < 0.0) store_real(g, x[c], i, 0.0);
        }
    }
    return REF_OK;
}

/* ---------------------------------------------------------------------------
 * O5 / a8. One time step in the paper's loop order setrho -> (field_solver: not
 * considered) -> accel -> push, preceded by the sort
 * (reading R6): sort(in) -> out; rho from out at x(t); then out advanced in place.
 * do_sort = 0: the particles are copied in their current order (perm = identity,
 * cell_offsets untouched).
 * ------------------------------------------------------------------------- */
int pic_ref_step(const pic_ref_grid *g, int64_t n,
                 const void *const xin[3], const void *const vin[3], const void *win,
                 void *const xout[3], void *const vout[3], void *wout,
                 int32_t *perm, int32_t *cell_offsets, double *rho,
                 const void *const E[3], double dt, double qm, int do_sort)
{
    if (!grid_ok(g) || n < 0) return REF_BAD_ARG;
    if (do_sort) {
        int rc = pic_ref_sort(g, n, xin, vin, win, xout, vout, wout, perm, cell_offsets);
        if (rc) return rc;
    } else {
        size_t s = g->dtype ? 8 : 4;
        for (int c = 0; c < g->dim; ++c) {
            memcpy(xout[c], xin[c], s * (size_t)n);
            memcpy(vout[c], vin[c], s * (size_t)n);
        }
        memcpy(wout, win, s * (size_t)n);
        if (perm) for (int64_t i = 0; i < n; ++i) perm[i] = (int32_t)i;
    }
    int rc = pic_ref_deposit(g, n, (const void *const *)xout, wout, rho);
    if (rc) return rc;
    return pic_ref_push(g, n, xout, vout, E, dt, qm);
}
