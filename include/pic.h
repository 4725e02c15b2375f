/*
 * pic.h -- C-ABI boundary of the B200-native particle hot path of PIC_ENGINE
 * (arXiv 1603.02886): per-step sort by cell key, B-spline charge deposit, field
 * gather + accel + push.  Implementation: paper_1603_02886_b200/csrc (CUDA, sm_100a).
 *
 * Citations are lines of /root/reference/PAPER.md plus the section they fall in;
 * R<n> are the readings of silent/garbled passages listed in DESIGN.md.
 *
 * Conventions common to every entry point
 * ---------------------------------------
 *  - Pointers inside pic_particles_t, rho, E[], perm, cell_offsets and ws are DEVICE
 *    pointers unless an argument says "host".  pic_grid_t / pic_particles_t themselves
 *    are small host structs passed by pointer and read before the call returns.
 *  - Particles are a contiguous structure of arrays, one array per attribute
 *    ("part_att(num_part, natt)", SoA, section 3.1): x[c], v[c] for
 *    c < dim, and the weight w (R2).  Element type = grid->dtype (float or double).
 *    Unused components (c >= dim) are ignored and may be NULL.
 *  - Grid arrays are x fastest: node (jx,jy,jz) at jx + n[0]*(jy + n[1]*jz)
 *    ("rho[(..)+nx*(..)+nx*ny*iz2]", App. B).  n nodes per dimension,
 *    periodic, node j at coordinate j*h (R4).  E is three separate grids
 *    (section 4.2).
 *  - Ownership: the caller owns every buffer, including the workspace; the library
 *    allocates nothing, frees nothing and keeps no particle or grid state between calls
 *    (the only per-thread state is the launch counter and the optional phase-event hook below).
 *    What carries over from one call to the next lives in the caller's buffers: cell_offsets (an order
 *    hint, see pic_sort) and, for PIC_SORT_CHAINED, the workspace (see pic_step).
 *  - Execution: all work is enqueued on `stream` (a cudaStream_t passed as void*);
 *    no host synchronisation and no host<->device copy happens inside ("data transfers
 *    ... kept to a minimum").  Results are valid once the stream is synced.
 *  - Errors: every function returns a pic_status_t.  Arguments are validated on the
 *    host BEFORE any launch: dim in {2,3}; order in {1,2,3}; n[c] >= order+1 for
 *    c < dim; prod n < 2^31; h[c] > 0; 0 <= N < 2^30; non-null pointers aligned to 16 bytes (arrays
 *    of an empty particle set may be NULL); workspace >= pic_workspace_bytes.  A failed launch gives PIC_ERR_CUDA.
 *  - Precondition, not checked: 0 <= x[c] < n[c]*h[c].  Cell indices are clamped
 *     and stencil nodes are folded mod n, so out-of-range positions can
 *    never cause an out-of-bounds access, only a meaningless deposit.
 */
#ifndef PIC_H_
#define PIC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { PIC_F32 = 0, PIC_F64 = 1 } pic_dtype_t;

typedef enum {
    PIC_OK = 0,
    PIC_ERR_INVALID_ARG = -1,   /* null/misaligned pointer, bad dim/order/n/h/N */
    PIC_ERR_UNSUPPORTED = -2,   /* valid request this build has no kernel for */
    PIC_ERR_WORKSPACE = -3,     /* ws_bytes < pic_workspace_bytes() */
    PIC_ERR_CUDA = -4,          /* launch failure; see cudaGetLastError() */
    PIC_ERR_TOO_LARGE = -5      /* pic_deposit_static: the grid has more than PIC_DEPOSIT_STATIC_MAX_NODES nodes */
} pic_status_t;

/* How the particle array handed to pic_deposit / pic_push is ordered. */
typedef enum {
    PIC_ORDER_UNSORTED = 0,     /* arbitrary order: threads-on-particles with global atomics
                                   (setrho 3.3.4) */
    PIC_ORDER_SORTED = 1,       /* sorted by cell key and cell_offsets describes it exactly */
    PIC_ORDER_STALE = 2         /* sorted some steps ago: mostly local, exactness still required */
} pic_order_t;

typedef struct {
    int32_t dim;        /* 2 or 3 */
    int32_t n[3];       /* cells = nodes per dimension; n[2] ignored when dim == 2 */
    double  h[3];       /* grid spacing; box length L[c] = n[c]*h[c]; origin 0 */
    int32_t order;      /* B-spline degree p: 1 (the paper's linear splines), 2, 3 (R1) */
    int32_t dtype;      /* pic_dtype_t of particles, rho and E */
} pic_grid_t;

typedef struct {
    void   *x[3];       /* positions  x[c][N], device */
    void   *v[3];       /* velocities v[c][N], device */
    void   *w;          /* weights    w[N],    device */
    int64_t n;          /* number of particles N */
} pic_particles_t;

/* Bytes of device workspace that pic_sort / pic_deposit / pic_step need for N particles
 * on this grid (a multiple of 256).  Pure host computation. */
int pic_workspace_bytes(const pic_grid_t *grid, int64_t n, size_t *bytes /* host, out */);

/*
 * pic_sort -- stable counting sort of the particles by cell key (rows a1-a4).
 *   key_i = c_x + n_x*(c_y + n_y*c_z), c = clamp(floor(x/h), 0, n-1): the particle's target
 *   bucket, one cell per bucket, bins x fastest (section 3.2; 489-497 App. B).
 *   histogram -> exclusive prefix sum -> scatter (Alg. 2 lines 1-5).
 *   The paper's atomic-counter scatter leaves the order inside a bucket arbitrary; here ties keep
 *   ascending source index, so perm is unique (R7).  floor(x/h) is an IEEE division in the storage
 *   dtype (R13).
 * in  : particles in any order (read only).
 * out : the same particles grouped by cell, out_a[j] = in_a[perm[j]] bit for bit.  Out of place
 *       (PAPER.md:120-122); `out` must not alias `in` -- the caller ping-pongs instead of the
 *       paper's copy-back.
 * perm[N]          : int32, perm[j] = source index of the particle now at position j (R9).
 * cell_offsets[C+1]: int32, IN/OUT.  On return: particles of cell k occupy [cell_offsets[k], cell_offsets[k+1]).
 *       On ENTRY the array is READ as an optional order hint: if it holds the offsets of an earlier sort of
 *       these particles (in a time loop: the previous step's output) only the particles that have left their
 *       interval since are sorted ("pre-ordered particles", Alg. 2).  The result
 *       never depends on what the array holds -- any content, including uninitialised memory, gives the same
 *       perm and offsets, only slower -- but the memory must be readable; zero it where a tool such as
 *       compute-sanitizer initcheck is used.
 */
int pic_sort(const pic_grid_t *grid, const pic_particles_t *in, pic_particles_t *out,
             int32_t *perm, int32_t *cell_offsets, void *ws, size_t ws_bytes, void *stream);

/*
 * pic_deposit -- charge deposition, setrho (row a5; PAPER.md:79 step i, 200, 292-294 section 3.3.4,
 * CUDA kernel PAPER.md:479-526).
 *   rho[j] = h^-d * sum_i w_i * prod_c W_p(x_ic/h_c - j_c), (p+1)^d nodes per particle, periodic.
 *   p = 1 reproduces the paper's 8 trilinear products; w and 1/h^d are R2.
 * rho[C] is OVERWRITTEN (R10).  Summation order is unspecified (atomics): results agree with
 * the oracle to rounding, not bit for bit.
 * order/cell_offsets: PIC_ORDER_SORTED selects the per-cell path (thread-private sums, one global
 * reduction per node and cell run; "sorting is required");
 * cell_offsets may be NULL for UNSORTED.
 * ws: fp32 grids accumulate in a double-precision grid of the workspace (rounded once into rho), so
 * ws of at least pic_workspace_bytes() is REQUIRED when dtype == PIC_F32; fp64 grids accumulate in
 * rho itself and ws may be NULL.
 */
int pic_deposit(const pic_grid_t *grid, const pic_particles_t *p, int order_state,
                const int32_t *cell_offsets, void *rho, void *ws, size_t ws_bytes, void *stream);

/*
 * pic_deposit_static -- pic_deposit for callers that cannot allocate device memory: no workspace argument.
 *
 * Why it exists.  On an fp32 grid pic_deposit sums in a double-precision copy of the grid (rounded into rho once at the
 * end) and takes that copy from a caller-allocated workspace.  A caller that is only handed its input and output
 * buffers has nowhere to get one: a plug-in inside an application that owns the device heap, code on a latency budget
 * where cudaMalloc / cudaFree are ruled out because they may synchronise the device, or a process that starts after all
 * GPU memory went to pools.  For them the double grid is a fixed-size array INSIDE the library: every GPU that loads the
 * library carries PIC_DEPOSIT_STATIC_MAX_NODES doubles (16 MiB) of it until the process exits, used or not.
 *
 * What it computes.  rho[C] (overwritten) exactly as pic_deposit(grid, p, PIC_ORDER_UNSORTED, ...) does: the paper's
 * "threads on particles" deposit with atomic additions (setrho 3.3.4; formula and R2/R10 as for
 * pic_deposit), correct for any particle order; the two agree to the rounding of the double sums.  Only x[c] (c < dim)
 * and w of p are read.
 *
 * Limits and rules.
 *  - dtype must be PIC_F32.  PIC_F64 returns PIC_ERR_UNSUPPORTED: an fp64 grid sums in rho itself, so plain pic_deposit
 *    with ws = NULL already allocates nothing.
 *  - prod n <= PIC_DEPOSIT_STATIC_MAX_NODES (2^21 = a 128^3 grid), else PIC_ERR_TOO_LARGE and nothing is enqueued.
 *  - The call itself never calls cudaMalloc, cudaFree or a library routine that allocates; it enqueues one memset and
 *    two kernels on `stream`.
 *  - The FIRST call on each device looks up that device's address of the array (cudaGetSymbolAddress, with the device
 *    current; it may make the runtime load the library's code onto that device).  Make that first call during set-up,
 *    before any stream capture is open, with the device that `stream` belongs to current -- as for every call.
 *  - All calls on one device share the one array and find the previous call's sums in it; each call clears the part it
 *    uses first, on its stream.  Two calls that can run at the same time on the GPU (different streams without an
 *    ordering between them, or two host threads) RACE on the array and both get wrong densities.  Order them.
 */
#define PIC_DEPOSIT_STATIC_MAX_NODES (1 << 21)
int pic_deposit_static(const pic_grid_t *grid, const pic_particles_t *p, void *rho, void *stream);

/*
 * pic_deposit_nodes -- the same rho by the paper's COLLISION-FREE algorithm, "threads on splines" (setrho_splines,
 * PAPER.md:202-204 section 3.3.1 and Fig. 6; Fortran of App. B): the threads are
 * associated with the grid nodes, each node adds up the spline values of the particles of the cells around it, nothing
 * is written twice, no atomics.  Cost as the paper counts it, (Nx+d)(Ny+d)(Nz+d) Np/Nbuckets, with one cell per bucket.
 * p must be sorted by cell and cell_offsets[C+1] must be the offsets of that order (pic_sort's output).
 * The additions of a node happen in a FIXED order -- ascending position in the sorted array -- in double, every
 * operation rounded on its own: rho is bitwise reproducible from run to run, and it IS the particle-order double sum
 * of the definition (rounded once to float for fp32 grids).  pic_deposit gives the same numbers to rounding, faster.
 * If cell_offsets does not describe the order of p (checked on the device) the call still returns the correct rho,
 * computed by pic_deposit's any-order kernel, without the reproducibility.
 * ws: at least pic_workspace_bytes(), for both dtypes.  rho[C] is overwritten.
 */
int pic_deposit_nodes(const pic_grid_t *grid, const pic_particles_t *p, const int32_t *cell_offsets,
                      void *rho, void *ws, size_t ws_bytes, void *stream);

/*
 * pic_deposit_replicated -- the same rho by the paper's other collision-free algorithm, "threads on buckets with data
 * replication" (section 3.3.3, Fig. 7): the threads are associated with the buckets
 * (here: cells) of sorted particles, each sums its particles onto a LOCAL grid of its own -- the cell's nodes plus the guard
 * nodes its stencils reach -- kept in a temporary global array "without atomics in global memory"; in a second step
 * "threads are assigned to the grid and collect the data from the temporary variables".  No atomic operation anywhere
 * and a fixed order of additions (per cell in particle order, then the cells around a node in ascending order): bitwise
 * reproducible; equal to pic_deposit within rounding.  p sorted by cell, cell_offsets from pic_sort; if they do not
 * describe the order (checked on the device) the any-order kernel answers instead.
 * ws: pic_deposit_replicated_bytes() = pic_workspace_bytes() + (4 or 2)^dim doubles per cell.  rho[C] is overwritten.
 */
int pic_deposit_replicated_bytes(const pic_grid_t *grid, int64_t n, size_t *bytes /* host, out */);
int pic_deposit_replicated(const pic_grid_t *grid, const pic_particles_t *p, const int32_t *cell_offsets,
                           void *rho, void *ws, size_t ws_bytes, void *stream);

/*
 * pic_push -- field gather + accel + push in one pass (rows a6-a7; PAPER.md:82-83 steps iii-iv,
 * 86, 88; models PAPER.md:312, 316):
 *   E_i = sum_j E[j] * prod_c W_p(x_ic/h_c - j_c)   (same splines as the deposit)
 *   v_i += qm*dt*E_i          (field at the OLD position)
 *   x_i += dt*v_i             (the NEW velocity), then x -= L*floor(x/L); 0 <= x < L in storage.
 * x and v are updated in place; w is not read.  E[c][C] for c < dim, each a separate grid.
 */
int pic_push(const pic_grid_t *grid, pic_particles_t *p, int order_state,
             const int32_t *cell_offsets, const void *const E[3], double dt, double qm,
             void *stream);

/*
 * pic_step -- one time step of the hot path (row a8): sort (if do_sort) -> deposit at x(t) ->
 * accel -> push, the paper's loop order setrho -> accel -> push with the
 * field solve left out as in the paper and the re-sort of PAPER.md:100 placed first (R6).
 * out receives the particles in sorted order, advanced to t+1; rho is the density at t.
 * do_sort = PIC_SORT (1), or any other non-zero value except PIC_SORT_CHAINED: sort by the keys of the positions in
 *   `in`; cell_offsets is read on entry as a hint and overwritten, exactly as in pic_sort; `out` must not overlap `in`.
 * do_sort = PIC_SORT_CHAINED (3): the same result, for a time loop.  The caller states that `in` is, UNMODIFIED,
 *   the `out` of the previous pic_step(do_sort != 0) call made with this workspace.  That call's step kernel had
 *   every advanced position in registers and left the next keys, their histogram and the list of particles that
 *   changed cell in the workspace ("emission of next-step keys"), so this call's sort does not
 *   read the positions again.  What can be checked is checked on the device (same N, grid and array addresses; the
 *   workspace was not used by another sort or step in between): if it does not hold, the call behaves like
 *   PIC_SORT.  What cannot be checked is the caller's statement itself: particle data changed in place between
 *   the two calls gives a wrong order.  In a chain the hint is the workspace's own copy of the previous
 *   offsets; cell_offsets is only written.
 *   NOTHING ELSE MAY TOUCH THE WORKSPACE between two chained steps.  The signature that vouches for the emission is
 *   the first 256 bytes of the workspace, for every N and grid, and every other call of this library that is given
 *   a workspace ends the chain there (pic_sort*, pic_deposit* with a workspace, pic_field_solve, pic_step with
 *   do_sort = 0 or PIC_SORT, pic_step_buckets, pic_step_selfconsistent): the next PIC_SORT_CHAINED call then simply
 *   sorts like PIC_SORT.  Writes of the caller's own into the workspace are covered only as far as they hit those
 *   first bytes; past them they corrupt the emission unseen (wrong order, possibly out-of-bounds indices).
 * do_sort = 0: particles keep their order (out_a[j] = advanced in_a[j]; out may be the same arrays as
 * in); perm is not written and cell_offsets is not modified.  cell_offsets NULL says "no order at all": the any-order
 * kernels run (threads on particles, setrho 3.3.4).  cell_offsets non-NULL says "these particles
 * were sorted some steps ago": the step kernel then walks runs of equal cell key, which it finds from the
 * positions themselves (the array's contents are not read), and a particle that has drifted out of the run around
 * it is taken on its own (threads on particles).  The result is exact whatever the order really is.
 * This is config 5's "sort every 4 / 16 steps" arm.  On this hardware it is slower than
 * sorting every step: a particle that has left its cell since the last sort pays (p+1)^d global reductions and
 * uncoalesced field reads, a re-sort of the 15-25 % movers costs far less (numbers in DESIGN.md section 5.4).
 */
#define PIC_SORT 1
#define PIC_SORT_CHAINED 3
int pic_step(const pic_grid_t *grid, const pic_particles_t *in, pic_particles_t *out,
             int32_t *perm, int32_t *cell_offsets, void *rho, const void *const E[3],
             double dt, double qm, int do_sort, void *ws, size_t ws_bytes, void *stream);

/*
 * Buckets of several cells.  "Particles are sorted into buckets ... a bucket [is] one or more
 * grid cells" (section 3.2); the paper's experiment is the sweep over the number of buckets
 * (Fig. 9, 396-402 Fig. 14).  A bucket is a box of bucket[c] cells per dimension (1 <= bucket[c] <=
 * n[c]; the last bucket of a dimension is smaller when bucket[c] does not divide n[c]); there are
 * nb[c] = ceil(n[c] / bucket[c]) of them per dimension, ordered x fastest like the paper's bins ("ibin = bin %
 * nsplitx; jbin = bin / nsplitx", App. B):
 *     key_i = b_x + nb_x*(b_y + nb_y*b_z),  b_c = floor(cell_c / bucket[c]),  cell_c the clamped cell index of pic_sort.
 * bucket is a HOST array of 3 ints (entries c >= dim ignored).  bucket = (1,1,1) gives exactly pic_sort / pic_step(PIC_SORT).
 *
 * pic_bucket_count: B = prod nb[c] (host computation).
 * pic_sort_buckets: the stable counting sort of pic_sort with this key.  Particles of one bucket become contiguous and
 *   keep their source order inside it (R7; the paper leaves it arbitrary).  bucket_offsets[B+1] is IN/OUT exactly like
 *   pic_sort's cell_offsets (an optional order hint on entry; offsets of the buckets on return).  Workspace:
 *   pic_workspace_bytes() of the grid.
 * pic_step_buckets: sort by bucket, then deposit + gather + accel + push in one pass over the particles in bucket
 *   order; rho, out as in pic_step.  Buckets of at least 27 cells whose grid tile (bucket + stencil halo, rho in double
 *   and d field components) fits in 160 KB of shared memory take the paper's own CUDA design: a block per bucket stages the
 *   tile in shared memory, threads on particles add into it atomically and read the field from it, the tile is flushed
 *   with one global atomic per node (App. B).  Other buckets are walked as runs of equal
 *   CELL key (short inside a bucket, where the source order is kept), particles alone in their run going the
 *   threads-on-particles way (setrho 3.3.4).  The result is exact for every bucket size; one cell per
 *   bucket is by far the fastest on this hardware (the sweep is in profiles/ and DESIGN.md).
 *
 * pic_sort_buckets_inplace: the paper's preferred sort, "Bucketsort for pre-ordered particles, contiguous datastructure"
 *   (Alg. 2; text PAPER.md:190-196; "for the rest of this paper this sorting algorithm is
 *   considered"): IN PLACE, and only the misplaced particles move.  bucket_offsets
 *   (OUT only) = prefix sum of the key histogram; a particle is misplaced if its array position lies outside the region
 *   [offsets[key], offsets[key+1]) of its own key (l.6-17 of the listing); misplaced particles are copied to a buffer
 *   grouped by target bucket, their positions are the holes, grouped by region; buffer entry i goes into hole i
 *   (l.21-35).  The paper hands out buffer slots with atomic counters; here slots go in ascending array position on both
 *   sides (R24), so the result is unique.  NOT stable: particles already inside their region stay where they are.
 *   *moved (device int32, may be NULL) = number of misplaced particles.  ws: pic_sort_buckets_inplace_bytes() =
 *   pic_workspace_bytes() + all attributes of n particles (the particles_buffer at its largest).
 *   With one cell per bucket and many cells most particles count as misplaced after a single step, because every cell
 *   boundary shifts by the net flux of all cells below it; the sort pays off for large buckets.
 */
int pic_bucket_count(const pic_grid_t *grid, const int32_t bucket[3] /* host */, int64_t *count /* host, out */);
int pic_sort_buckets_inplace_bytes(const pic_grid_t *grid, int64_t n, size_t *bytes /* host, out */);
int pic_sort_buckets_inplace(const pic_grid_t *grid, const int32_t bucket[3] /* host */, pic_particles_t *p,
                             int32_t *bucket_offsets, int32_t *moved, void *ws, size_t ws_bytes, void *stream);
int pic_sort_buckets(const pic_grid_t *grid, const int32_t bucket[3] /* host */, const pic_particles_t *in,
                     pic_particles_t *out, int32_t *perm, int32_t *bucket_offsets, void *ws, size_t ws_bytes,
                     void *stream);
int pic_step_buckets(const pic_grid_t *grid, const int32_t bucket[3] /* host */, const pic_particles_t *in,
                     pic_particles_t *out, int32_t *perm, int32_t *bucket_offsets, void *rho,
                     const void *const E[3], double dt, double qm, void *ws, size_t ws_bytes, void *stream);

/*
 * The field solve and the closed loop.  Step ii of the paper's loop, "field_solver(): -Laplace(phi) =
 * rho" (section 3; "we solve Poisson's equation for computing the field potential phi"), with
 * periodic boundary conditions.  The paper leaves the step out ("not considered"); beyond the
 * equation everything is a reading (R21-R23): E = -grad(phi); the mean of rho is dropped (neutralising
 * background) and phi has zero mean; spectral discretisation on the node grid: with rho^ = DFT(rho) and
 * kappa_c(m) = 2 pi mt / L_c (mt = m for m <= n/2, m - n above), phi^ = rho^ / sum_c kappa_c^2 and E_c^ = -i kappa'_c phi^,
 * kappa' = kappa except 0 at the Nyquist index of an even n.
 *
 * pic_field_solve: rho[C] -> E[c][C] for c < dim and, if phi != NULL, phi[C]; all of the grid's dtype, x fastest; the
 *   arithmetic is double whatever the dtype.  Hand-written transforms (radix-2 for power-of-two n[c], the plain DFT sum
 *   otherwise); n[c] <= 4096, else PIC_ERR_UNSUPPORTED from every call of this group (the *_bytes ones included),
 *   returned before anything is enqueued or written.  ws: pic_field_solve_bytes().
 * pic_step_selfconsistent: one step of the closed loop i-iv: sort by cell (cell_offsets: in/out hint as in
 *   pic_sort), rho = deposit at x(t) (the reorder happens in the same pass), E = field_solve(rho) written to the
 *   caller's E[c], then v += qm dt E(x), x += dt v on the sorted particles.  out, perm, cell_offsets, rho as in pic_step.
 *   ws: pic_step_selfconsistent_bytes().
 */
int pic_field_solve_bytes(const pic_grid_t *grid, size_t *bytes /* host, out */);
int pic_field_solve(const pic_grid_t *grid, const void *rho, void *const E[3], void *phi /* may be NULL */,
                    void *ws, size_t ws_bytes, void *stream);
int pic_step_selfconsistent_bytes(const pic_grid_t *grid, int64_t n, size_t *bytes /* host, out */);
int pic_step_selfconsistent(const pic_grid_t *grid, const pic_particles_t *in, pic_particles_t *out,
                            int32_t *perm, int32_t *cell_offsets, void *rho, void *const E[3],
                            double dt, double qm, void *ws, size_t ws_bytes, void *stream);

/*
 * pic_step_host -- the same step on HOST buffers: copies `in`, E to the device, runs pic_step,
 * copies out, perm, cell_offsets, rho back and synchronises.  All pointers (including those
 * inside in/out) are host pointers; dev_ws is a DEVICE scratch buffer of at least
 * pic_step_host_bytes() bytes.  This is the end-to-end entry bench.py times ("e2e").
 */
int pic_step_host_bytes(const pic_grid_t *grid, int64_t n, size_t *bytes /* host, out */);
int pic_step_host(const pic_grid_t *grid, const pic_particles_t *in, pic_particles_t *out,
                  int32_t *perm, int32_t *cell_offsets, void *rho, const void *const E[3],
                  double dt, double qm, int do_sort, void *dev_ws, size_t dev_ws_bytes,
                  void *stream);

/*
 * pic_step_fields_host -- one step with the particles RESIDENT on the device and the grid quantities
 * on the host, the paper's arrangement: particle and grid arrays stay on the GPU ("present", PAPER.md:447;
 * transfers "kept to a minimum") while the field comes from a solver outside.
 * Copies E (HOST, each [C]) to the device, runs pic_step on the DEVICE arrays in / out / perm /
 * cell_offsets exactly as pic_step does, copies rho (HOST, [C]) back and synchronises the stream.
 * ws: DEVICE, at least pic_step_fields_host_bytes() bytes (the grids + the pic_step workspace).
 */
int pic_step_fields_host_bytes(const pic_grid_t *grid, int64_t n, size_t *bytes /* host, out */);
int pic_step_fields_host(const pic_grid_t *grid, const pic_particles_t *in, pic_particles_t *out,
                         int32_t *perm, int32_t *cell_offsets, void *rho /* host */,
                         const void *const E[3] /* host */, double dt, double qm, int do_sort,
                         void *ws, size_t ws_bytes, void *stream);

/* Number of kernels the last call of this thread enqueued (for bench.py's gpu_launches). */
int pic_last_launch_count(void);

/*
 * pic_set_phase_events -- optional per-phase timing.  `events` is a host array of `count`
 * cudaEvent_t handles (as void*) owned by the caller, or NULL/0 to switch the hook off.  While
 * set (per host thread), pic_sort / pic_deposit / pic_push / pic_step record events[k] on the
 * call's stream at the END of phase k (slots >= count are skipped):
 *   PIC_PHASE_BEGIN 0  before the first kernel      PIC_PHASE_KEYS   1  cell keys + histogram
 *   PIC_PHASE_SCAN  2  prefix sums                   PIC_PHASE_RADIX  3  stable scatter of (key,index)
 *   PIC_PHASE_REORDER 4 attribute reorder            PIC_PHASE_DEPOSIT 5 deposit
 *   PIC_PHASE_PUSH  6  gather + accel + push (or the fused deposit+push kernel)
 * Recording an event costs no synchronisation; bench.py uses this to time the dominant kernel.
 */
#define PIC_PHASE_BEGIN 0
#define PIC_PHASE_KEYS 1
#define PIC_PHASE_SCAN 2
#define PIC_PHASE_RADIX 3
#define PIC_PHASE_REORDER 4
#define PIC_PHASE_DEPOSIT 5
#define PIC_PHASE_PUSH 6
#define PIC_NUM_PHASES 7
int pic_set_phase_events(void *const *events /* host */, int count);

/* Static, human-readable text for a pic_status_t. */
const char *pic_strerror(int status);

#ifdef __cplusplus
}
#endif
#endif /* PIC_H_ */
