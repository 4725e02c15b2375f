// pic_common.cuh -- device-side helpers shared by the kernels of the CUDA path.
// Nothing here is shared with oracle/ (the CPU oracle has its own statement of everything).
//
// Citations: PAPER.md:NNN = line of /root/reference/PAPER.md; R<n> = DESIGN.md reading.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/pic.h"

namespace pic {

constexpr int kMaxPasses = 4;      // radix passes of 8 bits cover 32-bit keys
constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;

// Grid parameters in the storage precision T, passed to kernels by value.
template <typename T>
struct GridP {
    int n[3];        // nodes per dimension (n[2] = 1 in 2-D)
    T h[3];          // spacing
    T inv_h[3];      // 1/h (exact when h is a power of two)
    T L[3];          // box length n*h
    T inv_L[3];
    T inv_vol;       // 1 / prod h
    int hmul;        // 1: every h is a power of two, x*inv_h == x/h bit for bit
    double Ld[3];    // box length in double (advance_wrap)
    int bk[3];       // cells per bucket and dimension (sort key of pic_sort_buckets; 1 = one cell per bucket)
    int nbk[3];      // buckets per dimension = ceil(n / bk)
};

template <typename T>
inline GridP<T> make_gridp(const pic_grid_t& g, const int32_t* bucket = nullptr)
{
    GridP<T> p;
    double vol = 1.0;
    int hmul = 1;
    for (int c = 0; c < 3; ++c) {
        bool on = c < g.dim;
        p.n[c] = on ? g.n[c] : 1;
        double h = on ? g.h[c] : 1.0;
        p.h[c] = (T)h;
        p.inv_h[c] = (T)1 / p.h[c];
        double L = (double)p.n[c] * h;
        p.L[c] = (T)L;
        p.Ld[c] = L;
        p.inv_L[c] = (T)(1.0 / L);
        p.bk[c] = (on && bucket) ? bucket[c] : 1;
        p.nbk[c] = (p.n[c] + p.bk[c] - 1) / p.bk[c];
        if (on) {
            vol *= h;
            int e;
            double m = frexp((double)p.h[c], &e);
            if (m != 0.5) hmul = 0;
        }
    }
    p.inv_vol = (T)(1.0 / vol);
    p.hmul = hmul;
    return p;
}

// Particle arrays by value (device pointers).
template <typename T>
struct PartP {
    T* x[3];
    T* v[3];
    T* w;
};

template <typename T>
inline PartP<T> make_partp(const pic_particles_t& p)
{
    PartP<T> q;
    for (int c = 0; c < 3; ++c) { q.x[c] = (T*)p.x[c]; q.v[c] = (T*)p.v[c]; }
    q.w = (T*)p.w;
    return q;
}

// t = x/h by IEEE division in the storage precision (R13); the paper works in grid units,
// "ix = (int) x".  When h is a power of two the product is the same number.
template <typename T>
__device__ __forceinline__ T grid_coord(T x, T h, T inv_h, int hmul)
{
    return hmul ? x * inv_h : x / h;
}

// Clamped cell index: "if (ix<0) ix=0; if (ix>nx-1) ix=nx-1".
// floor() by a saturating round-down conversion (NaN -> 0), then an integer clamp: no branches.
__device__ __forceinline__ int floor_to_int(float t) { return __float2int_rd(t); }
__device__ __forceinline__ int floor_to_int(double t) { return __double2int_rd(t); }
template <typename T>
__device__ __forceinline__ int cell_index(T t, int n)
{
    return max(0, min(floor_to_int(t), n - 1));
}

// Sort key of a particle from its clamped cell indices.  BK = false: the cell key, x fastest (a1,
// PAPER.md:489-490).  BK = true: the key of its BUCKET, a box of bk[c] cells per dimension, buckets x fastest
// ("a bucket ... one or more grid cells"; "ibin = bin % nsplitx; jbin = bin / nsplitx",
// PAPER.md:487-490): key = b_x + nb_x (b_y + nb_y b_z), b_c = floor(cell_c / bk_c).
template <typename T, int D, bool BK>
__device__ __forceinline__ int sort_key(const GridP<T>& g, const int (&cell)[3])
{
    int k = 0, mul = 1;
#pragma unroll
    for (int c = 0; c < D; ++c) {
        k += mul * (BK ? cell[c] / g.bk[c] : cell[c]);
        mul *= BK ? g.nbk[c] : g.n[c];
    }
    return k;
}

// One-dimensional stencil of degree P: first (unfolded) node and the P+1 weights.
// xi = t - i0 in [0,1].  P = 1: (1-xi, xi), the factors of PAPER.md:509-519.
template <typename T, int P>
__device__ __forceinline__ void spline_weights(T t, int i0, int& first, T (&w)[P + 1])
{
    T xi = t - (T)i0;
    if (P == 1) {
        first = i0;
        w[0] = (T)1 - xi;
        w[1] = xi;
    } else if (P == 2) {
        int up = xi >= (T)0.5 ? 1 : 0;
        T d = xi - (T)up;
        first = i0 + up - 1;
        T a = (T)0.5 - d, b = (T)0.5 + d;
        w[0] = (T)0.5 * a * a;
        w[1] = (T)0.75 - d * d;
        w[P] = (T)0.5 * b * b;
    } else {
        T om = (T)1 - xi;
        T x2 = xi * xi;
        first = i0 - 1;
        w[0] = om * om * om * (T)(1.0 / 6.0);
        w[P] = x2 * xi * (T)(1.0 / 6.0);
        w[1] = (T)(2.0 / 3.0) - x2 + (T)0.5 * x2 * xi;
        w[P - 1] = (T)(1.0 / 6.0) + (T)0.5 * (xi + x2 - x2 * xi);
    }
}

// fold an index in [-n, 2n) into [0, n)
__device__ __forceinline__ int fold(int j, int n)
{
    j = j < 0 ? j + n : j;
    return j >= n ? j - n : j;
}

// Periodic wrap of a pushed position into [0, L) in the storage precision.
template <typename T>
__device__ __forceinline__ T wrap_periodic(T x, T L, T inv_L)
{
    if (x < (T)0 || x >= L) {
        x -= L * floor(x * inv_L);
        if (x < (T)0) x += L;
        if (x >= L) x -= L;
        if (!(x >= (T)0 && x < L)) x = (T)0;
    }
    return x;
}

// A particle that leaves [0, L) in this step: accel and push are redone in double precision, wrapped and
// rounded once, as O4 states them.  (In the storage precision the sum x + dt v loses the low bits of x as soon
// as the particle crosses several boxes; inside the box the plain storage-precision update is within half an
// ulp of L of this.)  Out of line: the call is rare.
template <typename T>
__device__ __noinline__ T advance_wrap(T x_old, T v_old, T e, double dt, double qmdt, double L)
{
    const double vn = (double)v_old + qmdt * (double)e;
    double xn = (double)x_old + dt * vn;
    xn -= L * floor(xn / L);
    T xs = (T)xn;
    if (!(xs >= (T)0 && xs < (T)L)) xs = (T)0;
    return xs;
}

#define PIC_CUDA_OK(expr)                          \
    do {                                           \
        if ((expr) != cudaSuccess) return PIC_ERR_CUDA; \
    } while (0)

// multiprocessors of the current device (grids of the grid-stride kernels are sized from it)
int sm_count();
// thread-local launch counter behind pic_last_launch_count()
void count_launch(int n = 1);
// records the caller's event for `phase` on `st` if pic_set_phase_events() installed one
void mark_phase(int phase, cudaStream_t st);

// positions per staging tile of the movers (k_classify: half a block; k_runs: one warp's range)
constexpr int kStageTile = 2048;

// What a step kernel leaves behind for the NEXT step's sort (row a8: "emission of next-step keys + histogram").
// The advanced position of slot j is in registers, so its next cell key costs a few instructions here instead of a
// pass over x[d] there.  Slot j lies in the interval of its present key in this step's cell_offsets -- which are the
// next sort's hint -- so "stays in its interval" is simply new key == present key, and "comes from below the
// interval of its new key" is new key > present key (the intervals are ordered by key): no offsets are read.
// The layout is k_classify's (pic_sort.cu): tiles of kStageTile positions = one warp's range here.
struct EmitP {
    uint32_t* pkey;          // [N] next key of every slot
    uint32_t* mask;          // [N/32] mover bits of every 32 slots
    uint32_t* mprefix;       // [N/32] movers before the word, within its tile
    uint32_t* stage_key;     // [N] movers of tile t, in slot order, from t*kStageTile on: next key ...
    uint32_t* stage_idx;     //     ... and slot
    int32_t* tile_count;     // [tiles] movers of the tile
    int32_t* cell_out;       // [C] particles that leave cell k                        (zeroed by the caller)
    unsigned long long* mover_in;   // [C] low word: movers into cell k; high word: those of them that come from below
};

// What identifies the particle set a chain of pic_step calls works on (see PIC_SORT_CHAINED in pic.h): written
// to the workspace after a step, compared with the next call's arguments on the device.
struct ChainSig {
    uint64_t magic;          // kChainMagic when a step has left its emission behind, else anything
    uint64_t n, cells, grid; // particles, cells, hash of the grid parameters
    uint64_t arr[7];         // the arrays that hold the particles (out of the step that wrote it = in of the next)
};
constexpr uint64_t kChainMagic = 0x50494332434841ull;     // "PIC2CHA"

// ---- launchers implemented in the .cu files (all enqueue on `st`) ------------------------
struct SortWs {
    uint32_t* keys[2];       // [N] movers' keys, ping-pong
    uint32_t* idx[2];        // [N] movers' positions, ping-pong
    uint32_t* pkey;          // [N] key of every position
    uint32_t* mask;          // [N/32 + 2] mover bit of every position
    uint32_t* mprefix;       // [N/32 + 2] movers before each 32-position word
    int32_t* old_off;        // [C+1] the hint: cell_offsets as found on entry
    int32_t* mover_off;      // [C+1] exclusive scan of mover_count
    int32_t* cell_base;      // [C]   where the stayers of a cell start in perm (see k_cell_base)
    int32_t* tile_count;     // [classify tiles] movers per tile
    int32_t* tile_base;      // [classify tiles + 1] exclusive scan of tile_count
    uint32_t* lookback;      // [passes][radix tiles][kRadix]
    int32_t* cell_count;     // [C+1] histogram of the keys              (hist region: these three)
    int32_t* mover_count;    // [C+1] histogram of the movers' keys
    int32_t* mover_lo;       // [C+1] movers into a cell from below its hint interval
    uint32_t* digit_hist;    // [kMaxPasses][kRadix]                      (zero region from here ...)
    uint32_t* scan_status;   // [2][scan tiles]
    uint32_t* cls_status;    // [scan tiles of the classify tiles]
    uint32_t* counters;      // [64] tile tickets, number of movers, hint and chain flags  (... to here)
    uint32_t* gate;          // one word of counters: 1 = more than half of the particles are movers (set by the sort)
    uint32_t* stray_count;   // one word of counters: particles the step kernel has set aside (zeroed with the counters)
    uint32_t* stray_list;    // [N] their slots (= idx[0]: free once perm is written)
    void* rec_scratch;       // 32 N bytes (keys, idx, pkey arrays: free once perm is written; + 12 N) for launch_reorder_records
    double* racc;            // [C] double accumulation grid of the deposit (not in the zero region)
    int32_t* prev_off;       // [C+1] cell_offsets as the last sort of a chain wrote them (the next one's hint)
    ChainSig* chain_sig;     // what that step worked on
    EmitP emit;              // where a step kernel leaves the next sort's inputs
    void* hist_begin;        // cell_count, mover_count, mover_lo: zeroed before k_classify, or in a chain formed from the emitted counters (k_hint_hist)
    size_t hist_bytes;
    void* emit_begin;        // emit.cell_out, emit.mover_in: zeroed before an emitting step kernel
    size_t emit_bytes;
    void* zero_begin;        // region that must be zero before a sort
    size_t zero_bytes;
    int passes, bits_per_pass, key_bits;
    int64_t radix_tiles, scan_tiles, cls_tiles, stage_tiles;
    int64_t nkeys;           // number of sort keys: cells, or buckets
    const int32_t* bucket;   // host: cells per bucket and dimension, or NULL (one cell per bucket)
};

size_t sort_ws_bytes(const pic_grid_t& g, int64_t n);
// bucket != NULL (host, bucket[c] cells per dimension): the sort key is the bucket, not the cell (pic_sort_buckets)
int carve_sort_ws(const pic_grid_t& g, int64_t n, void* ws, size_t ws_bytes, SortWs& out, const int32_t* bucket = nullptr);

// reorder = false: only perm and cell_offsets are produced (out is not written).  chained: the caller says that
// `in` is the unmodified output of the previous pic_step on this workspace (checked on the device against the
// workspace's ChainSig): keys, histograms and the stayer/mover split are then the ones that step emitted.
int launch_sort(const pic_grid_t& g, const pic_particles_t& in, pic_particles_t& out, int32_t* perm,
                int32_t* cell_offsets, const SortWs& ws, bool reorder, bool chained, cudaStream_t st);
// Alg. 2: sort in place by moving only the misplaced particles (ws carved with the bucket shape; buffer: A arrays of n)
int launch_sort_inplace(const pic_grid_t& g, const pic_particles_t& p, int32_t* offsets, const SortWs& ws, void* buffer,
                        int32_t* moved, cudaStream_t st);
int launch_chain_commit(const pic_grid_t& g, const pic_particles_t& out, const SortWs& ws, cudaStream_t st);
int launch_deposit(const pic_grid_t& g, const pic_particles_t& p, int order_state,
                   const int32_t* cell_offsets, void* rho, double* racc, cudaStream_t st);
int launch_push(const pic_grid_t& g, pic_particles_t& p, int order_state, const int32_t* cell_offsets,
                const void* const E[3], double dt, double qm, cudaStream_t st);
// deposit at x(t) + gather + accel + push in ONE kernel over particles in cell order: in place on p
// (perm == NULL), or reading particle perm[j] of src and writing slot j of p (the sort's reorder fused into
// the same pass).  With perm, *ws.gate (written by the sort: 1 = most particles move) chooses on the device
// between that one pass and reorder-then-in-place; without perm, *ws.stray_count is zeroed here.  Lone
// particles go through ws.stray_list to a threads-on-particles kernel.
// cell_sorted = false (with perm): perm groups the particles by bucket only (pic_step_buckets); nothing is emitted.
int launch_fused(const pic_grid_t& g, const pic_particles_t& src, pic_particles_t& p, const int32_t* perm,
                 const SortWs& ws, void* rho, const void* const E[3], double dt, double qm, cudaStream_t st,
                 bool cell_sorted = true, const int32_t* key_offsets = nullptr);
// the collision-free deposit with a fixed order of additions (pic_nodes.cu); p sorted by cell as cell_offsets says
int launch_deposit_nodes(const pic_grid_t& g, const pic_particles_t& p, const int32_t* cell_offsets, void* rho,
                         const SortWs& ws, cudaStream_t st);
// periodic Poisson solve (pic_field.cu): rho -> E[c] (and phi if not NULL), all [C] of the grid's dtype; ws: field_ws_bytes
size_t field_ws_bytes(const pic_grid_t& g);
// PIC_OK, or PIC_ERR_UNSUPPORTED if an axis is longer than this build's transforms take (n[c] <= 4096): checked by the
// entry points before anything is enqueued
int field_supported(const pic_grid_t& g);
int launch_field_solve(const pic_grid_t& g, const void* rho, void* const E[3], void* phi, void* ws, cudaStream_t st);
// the closed loop i-iv: deposit along perm (+ reorder into p), field solve, gather + accel + push in place
int launch_selfconsistent(const pic_grid_t& g, const pic_particles_t& src, pic_particles_t& p, const int32_t* perm,
                          const SortWs& ws, void* rho, void* const E[3], void* field_ws, double dt, double qm, cudaStream_t st);
// deposit by replication (setrho 3.3.3): per-cell local grids in `slab` (replicated_slab_bytes), then assembly per node
size_t replicated_slab_bytes(const pic_grid_t& g);
int launch_deposit_replicated(const pic_grid_t& g, const pic_particles_t& p, const int32_t* cell_offsets, void* rho,
                              const SortWs& ws, void* slab, cudaStream_t st);
// out_a[j] = in_a[perm[j]] for every attribute; runs only if *gate == want (gate may be NULL)
int launch_reorder(const pic_grid_t& g, const pic_particles_t& in, const pic_particles_t& out, const int32_t* perm,
                   const uint32_t* gate, uint32_t want, cudaStream_t st);
// the same through 32-byte records of interleaved attributes (for a nearly random perm); scratch: 32 N bytes
int launch_reorder_records(const pic_grid_t& g, const pic_particles_t& in, const pic_particles_t& out, const int32_t* perm,
                           void* scratch, const uint32_t* gate, uint32_t want, cudaStream_t st);

}  // namespace pic
