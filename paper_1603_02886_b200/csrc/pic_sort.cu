// pic_sort.cu -- stable counting sort of the particles by cell key (rows a1-a4 of the hot path).
//
// The paper sorts with histogram -> prefix sum -> atomic-counter scatter (section 3.2,
// Alg. 2 lines 1-5 PAPER.md:207-212) and notes that hand-written CUDA histogram and prefix-sum
// kernels were worth a factor 2.  The atomic scatter is not stable; this
// build needs the unique stable permutation (R7), so the scatter is an LSD radix sort of
// (key, source index) pairs, each pass a one-sweep partition: warp-aggregated ranking, per-tile
// digit counts chained by decoupled look-back, coalesced scatter from a shared-memory staging
// tile.  The full-key histogram and its exclusive scan give cell_offsets.
//
// Kernels:  k_keys_hist      x[d] -> key, full-key histogram (run-aggregated atomics), digit histograms
//           k_scan_cells     count[C] -> cell_offsets[C+1]   (single pass, decoupled look-back)
//           k_scan_digits    digit histograms -> exclusive global digit offsets
//           k_radix_pass     one stable partition by an 8-bit digit
//           k_reorder        out_a[j] = in_a[perm[j]] for every attribute
#include <cmath>

#include "pic_common.cuh"

namespace pic {

static inline size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

// ----------------------------------------------------------------------------- tile shapes
constexpr int kRadixThreads = 256;
constexpr int kRadixIPT = 16;
constexpr int kRadixTile = kRadixThreads * kRadixIPT;      // 4096 pairs per tile
constexpr int kRadixWarps = kRadixThreads / 32;

constexpr int kScanThreads = 256;
constexpr int kScanIPT = 8;
constexpr int kScanTile = kScanThreads * kScanIPT;         // 2048 counts per tile

constexpr uint32_t kFlagAgg = 1u << 30, kFlagPrefix = 2u << 30, kValMask = (1u << 30) - 1;

__device__ __forceinline__ uint32_t ld_volatile(const uint32_t* p)
{
    return *reinterpret_cast<const volatile uint32_t*>(p);
}
__device__ __forceinline__ void st_volatile(uint32_t* p, uint32_t v)
{
    *reinterpret_cast<volatile uint32_t*>(p) = v;
}

// ----------------------------------------------------------------------------- keys + histograms
// a1: key = c_x + n_x*(c_y + n_y*c_z) (x fastest), clamped cell index
// (PAPER.md:493-497).  a2: count[key]++ -- consecutive lanes holding the same key (the common
// case once the particles are pre-ordered) are merged into one atomic per run.
template <typename T, int D>
__global__ void __launch_bounds__(256) k_keys_hist(PartP<T> p, GridP<T> g, int64_t n, uint32_t* __restrict__ key_out,
                                                   int32_t* __restrict__ cell_count)
{
    const unsigned lane = threadIdx.x & 31;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t n_round = (n + 31) & ~(int64_t)31;          // keep warps converged for the shuffles
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_round; i += stride) {
        const bool valid = i < n;
        uint32_t key = 0xFFFFFFFFu;
        if (valid) {
            int k = 0, mul = 1;
#pragma unroll
            for (int c = 0; c < D; ++c) {
                T t = grid_coord(p.x[c][i], g.h[c], g.inv_h[c], g.hmul);
                k += mul * cell_index(t, g.n[c]);
                mul *= g.n[c];
            }
            key = (uint32_t)k;
            key_out[i] = key;
        }
        // run-length aggregation inside the warp
        uint32_t prev = __shfl_up_sync(0xFFFFFFFFu, key, 1);
        bool head = (lane == 0) || (prev != key);
        unsigned heads = __ballot_sync(0xFFFFFFFFu, head);
        if (head && valid) {
            unsigned above = heads & ~((2u << lane) - 1);      // heads strictly above this lane
            int next = above ? __ffs(above) - 1 : 32;
            atomicAdd(&cell_count[key], next - (int)lane);
        }
    }
}

// ----------------------------------------------------------------------------- exclusive scan of the cell counts
// a3: cell_offsets[k] = sum_{k'<k} count[k'], cell_offsets[C] = N ("prefix sum").
// Single pass: each tile publishes its aggregate, then looks back over its predecessors.
// The per-pass digit histograms of the radix sort are summed here from the cell counts
// (C cells instead of N particles).
__global__ void __launch_bounds__(kScanThreads) k_scan_cells(const int32_t* __restrict__ count, int32_t* __restrict__ offsets,
                                                              int C, uint32_t* status, uint32_t* tile_counter,
                                                              uint32_t* __restrict__ digit_hist, int passes, int bits)
{
    __shared__ uint32_t s_warp[kScanThreads / 32];
    __shared__ uint32_t s_tile, s_excl;
    __shared__ uint32_t s_hist[kMaxPasses][kRadix];
    if (threadIdx.x == 0) s_tile = atomicAdd(tile_counter, 1u);
    for (int i = threadIdx.x; i < kMaxPasses * kRadix; i += kScanThreads) (&s_hist[0][0])[i] = 0;
    __syncthreads();
    const int tile = (int)s_tile;
    const int base = tile * kScanTile + threadIdx.x * kScanIPT;
    const unsigned lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    uint32_t v[kScanIPT];
    uint32_t sum = 0;
#pragma unroll
    for (int k = 0; k < kScanIPT; ++k) {
        v[k] = (base + k < C) ? (uint32_t)count[base + k] : 0u;
        sum += v[k];
    }
    {
        const uint32_t mask = (1u << bits) - 1;
        for (int q = 0; q < passes; ++q) {
#pragma unroll
            for (int k = 0; k < kScanIPT; ++k)
                if (v[k]) atomicAdd(&s_hist[q][((uint32_t)(base + k) >> (q * bits)) & mask], v[k]);
        }
    }
    // block-wide exclusive scan of the per-thread sums
    uint32_t inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
        if (lane >= (unsigned)o) inc += t;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    uint32_t warp_off = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) {
        uint32_t t = s_warp[w];
        if (w < (int)warp) warp_off += t;
        total += t;
    }
    uint32_t excl_thread = warp_off + inc - sum;

    // decoupled look-back, done by warp 0
    if (warp == 0) {
        if (lane == 0) st_volatile(&status[tile], (tile == 0 ? kFlagPrefix : kFlagAgg) | total);
        uint32_t excl = 0;
        int look = tile - 1;
        while (look >= 0) {
            int t = look - (int)lane;
            uint32_t s;
            do {
                s = (t >= 0) ? ld_volatile(&status[t]) : kFlagPrefix;
            } while (__any_sync(0xFFFFFFFFu, (s >> 30) == 0));
            unsigned pref = __ballot_sync(0xFFFFFFFFu, (s >> 30) == 2);
            int stop = pref ? __ffs(pref) - 1 : 31;            // nearest predecessor with an inclusive prefix
            uint32_t contrib = ((int)lane <= stop) ? (s & kValMask) : 0u;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) contrib += __shfl_xor_sync(0xFFFFFFFFu, contrib, o);
            excl += contrib;
            if (pref) break;
            look -= 32;
        }
        if (lane == 0) {
            if (tile != 0) st_volatile(&status[tile], kFlagPrefix | (excl + total));
            s_excl = excl;
        }
    }
    __syncthreads();
    uint32_t run = s_excl + excl_thread;
#pragma unroll
    for (int k = 0; k < kScanIPT; ++k) {
        if (base + k < C) offsets[base + k] = (int32_t)run;
        run += v[k];
        if (base + k == C - 1) offsets[C] = (int32_t)run;
    }
    for (int i = threadIdx.x; i < passes * kRadix; i += kScanThreads) {
        uint32_t c = (&s_hist[0][0])[i];
        if (c) atomicAdd(&digit_hist[i], c);
    }
}

// exclusive scan of each pass's 256-bin digit histogram, in place (one block per pass)
__global__ void __launch_bounds__(kRadix) k_scan_digits(uint32_t* digit_hist)
{
    __shared__ uint32_t s_warp[kRadix / 32];
    uint32_t* h = digit_hist + blockIdx.x * kRadix;
    const unsigned lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t c = h[threadIdx.x], inc = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
        if (lane >= (unsigned)o) inc += t;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    uint32_t off = 0;
    for (int w = 0; w < (int)warp; ++w) off += s_warp[w];
    h[threadIdx.x] = off + inc - c;
}

// ----------------------------------------------------------------------------- one radix pass
// Stable partition of (key, idx) pairs by digit (key >> shift) & mask (at most 8 bits).  Tile-local order is
// (warp, round, lane) = ascending input position, so equal digits keep their input order.
// idx_in == nullptr: idx is the input position (first pass).  keys_out == nullptr: keys are
// not needed any more (last pass).
__global__ void __launch_bounds__(kRadixThreads)
k_radix_pass(const uint32_t* __restrict__ keys_in, const uint32_t* __restrict__ idx_in,
             uint32_t* __restrict__ keys_out, uint32_t* __restrict__ idx_out, int64_t n, int shift, uint32_t mask,
             const uint32_t* __restrict__ digit_offsets, uint32_t* tile_counter, uint32_t* lookback)
{
    __shared__ uint32_t s_cnt[kRadixWarps][kRadix];   // per-warp digit counters -> per-warp bases
    __shared__ uint32_t s_start[kRadix];              // tile-local start of each digit
    __shared__ uint32_t s_base[kRadix];               // global address of local position 0 of each digit
    __shared__ uint32_t s_keys[kRadixTile];
    __shared__ uint32_t s_idx[kRadixTile];
    __shared__ uint32_t s_wsum[kRadixWarps];
    __shared__ uint32_t s_tile;

    const unsigned tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(tile_counter, 1u);
    for (int i = tid; i < kRadixWarps * kRadix; i += kRadixThreads) (&s_cnt[0][0])[i] = 0;
    __syncthreads();
    const int64_t tile = s_tile;
    const int64_t tile_base = tile * kRadixTile;
    const int tile_valid = (n - tile_base < (int64_t)kRadixTile) ? (int)(n - tile_base) : kRadixTile;

    // load, warp-striped: item r of this lane sits at warp*512 + r*32 + lane within the tile
    uint32_t key[kRadixIPT], val[kRadixIPT];
    uint16_t rank[kRadixIPT];
    const int wbase = warp * 32 * kRadixIPT + lane;
#pragma unroll
    for (int r = 0; r < kRadixIPT; ++r) {
        int loc = wbase + r * 32;
        bool ok = loc < tile_valid;
        key[r] = ok ? keys_in[tile_base + loc] : 0xFFFFFFFFu;
        val[r] = ok ? (idx_in ? idx_in[tile_base + loc] : (uint32_t)(tile_base + loc)) : 0u;
    }
    // warp-aggregated ranking: lanes with the same digit elect a leader that bumps the warp's counter
    const unsigned lt = (1u << lane) - 1;
#pragma unroll
    for (int r = 0; r < kRadixIPT; ++r) {
        uint32_t d = (key[r] >> shift) & mask;
        unsigned peers = __match_any_sync(0xFFFFFFFFu, d);
        int leader = __ffs(peers) - 1;
        uint32_t old = 0;
        if ((int)lane == leader) {
            old = s_cnt[warp][d];
            s_cnt[warp][d] = old + __popc(peers);
        }
        old = __shfl_sync(0xFFFFFFFFu, old, leader);
        rank[r] = (uint16_t)(old + __popc(peers & lt));
        __syncwarp();
    }
    __syncthreads();

    // per digit (thread d): exclusive scan over warps, tile total, look-back across tiles
    {
        const unsigned d = tid;            // kRadixThreads == kRadix
        uint32_t run = 0;
#pragma unroll
        for (int w = 0; w < kRadixWarps; ++w) {
            uint32_t c = s_cnt[w][d];
            s_cnt[w][d] = run;
            run += c;
        }
        const uint32_t total = run;
        // the padding keys of a ragged last tile all carry the highest digit and rank last; they are
        // never published (no tile follows) and never written (position >= tile_valid)
        uint32_t* my = lookback + tile * kRadix + d;
        st_volatile(my, (tile == 0 ? kFlagPrefix : kFlagAgg) | total);

        // tile-local exclusive scan over digits
        uint32_t inc = total;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
            if (lane >= (unsigned)o) inc += t;
        }
        if (lane == 31) s_wsum[warp] = inc;
        __syncthreads();
        uint32_t off = 0;
#pragma unroll
        for (int w = 0; w < kRadixWarps; ++w) off += (w < (int)warp) ? s_wsum[w] : 0u;
        const uint32_t start = off + inc - total;
        s_start[d] = start;

        uint32_t excl = 0;
        for (int64_t t = tile - 1; t >= 0; --t) {
            uint32_t s;
            do { s = ld_volatile(lookback + t * kRadix + d); } while ((s >> 30) == 0);
            excl += s & kValMask;
            if ((s >> 30) == 2) break;
        }
        if (tile != 0) st_volatile(my, kFlagPrefix | (excl + total));
        s_base[d] = digit_offsets[d] + excl - start;
    }
    __syncthreads();

    // scatter into the staging tile in sorted order
#pragma unroll
    for (int r = 0; r < kRadixIPT; ++r) {
        uint32_t d = (key[r] >> shift) & mask;
        uint32_t q = s_start[d] + s_cnt[warp][d] + rank[r];
        s_keys[q] = key[r];
        s_idx[q] = val[r];
    }
    __syncthreads();
    // coalesced write-out: consecutive local positions of one digit are consecutive in global memory
    for (int q = tid; q < tile_valid; q += kRadixThreads) {
        uint32_t k = s_keys[q];
        uint32_t dst = s_base[(k >> shift) & mask] + q;
        if (keys_out) keys_out[dst] = k;
        idx_out[dst] = s_idx[q];
    }
}

// ----------------------------------------------------------------------------- reorder
// a4: out_a[j] = in_a[perm[j]] for all attributes, bit for bit; coalesced writes, gathered reads.
template <typename T, int D>
__global__ void __launch_bounds__(256) k_reorder(PartP<T> in, PartP<T> out, const int32_t* __restrict__ perm, int64_t n)
{
    int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const int64_t i = perm[j];
    T x[D], v[D];
#pragma unroll
    for (int c = 0; c < D; ++c) { x[c] = in.x[c][i]; v[c] = in.v[c][i]; }
    T w = in.w[i];
#pragma unroll
    for (int c = 0; c < D; ++c) { out.x[c][j] = x[c]; out.v[c][j] = v[c]; }
    out.w[j] = w;
}

// ----------------------------------------------------------------------------- host side
static int key_bits_of(const pic_grid_t& g)
{
    int64_t C = 1;
    for (int c = 0; c < g.dim; ++c) C *= g.n[c];
    int b = 1;
    while (((int64_t)1 << b) < C) ++b;
    return b;
}

static int64_t cells_of(const pic_grid_t& g)
{
    int64_t C = 1;
    for (int c = 0; c < g.dim; ++c) C *= g.n[c];
    return C;
}

struct SortLayout {
    size_t keys0, keys1, idx0, idx1, zero_begin, cell_count, digit_hist, scan_status, counters, lookback, zero_end, racc, total;
    int passes, bits, key_bits;
    int64_t radix_tiles, scan_tiles;
};

static SortLayout sort_layout(const pic_grid_t& g, int64_t n)
{
    SortLayout L;
    const int64_t C = cells_of(g);
    L.key_bits = key_bits_of(g);
    L.passes = (L.key_bits + kRadixBits - 1) / kRadixBits;
    L.bits = (L.key_bits + L.passes - 1) / L.passes;
    L.radix_tiles = (n + kRadixTile - 1) / kRadixTile;
    L.scan_tiles = (C + kScanTile - 1) / kScanTile;
    size_t off = 0;
    const size_t nb = align256(sizeof(uint32_t) * (size_t)(n > 0 ? n : 1));
    L.keys0 = off; off += nb;
    L.keys1 = off; off += nb;
    L.idx0 = off; off += nb;
    L.idx1 = off; off += nb;
    L.zero_begin = off;
    L.cell_count = off; off += align256(sizeof(int32_t) * (size_t)C);
    L.digit_hist = off; off += align256(sizeof(uint32_t) * kMaxPasses * kRadix);
    L.scan_status = off; off += align256(sizeof(uint32_t) * (size_t)L.scan_tiles);
    L.counters = off; off += 256;
    L.lookback = off; off += align256(sizeof(uint32_t) * (size_t)L.passes * (size_t)(L.radix_tiles > 0 ? L.radix_tiles : 1) * kRadix);
    L.zero_end = off;
    L.racc = off; off += align256(sizeof(double) * (size_t)C);
    L.total = off;
    return L;
}

size_t sort_ws_bytes(const pic_grid_t& g, int64_t n) { return sort_layout(g, n).total; }

int carve_sort_ws(const pic_grid_t& g, int64_t n, void* ws, size_t ws_bytes, SortWs& o)
{
    SortLayout L = sort_layout(g, n);
    if (ws_bytes < L.total) return PIC_ERR_WORKSPACE;
    char* b = (char*)ws;
    o.keys[0] = (uint32_t*)(b + L.keys0);
    o.keys[1] = (uint32_t*)(b + L.keys1);
    o.idx[0] = (uint32_t*)(b + L.idx0);
    o.idx[1] = (uint32_t*)(b + L.idx1);
    o.cell_count = (int32_t*)(b + L.cell_count);
    o.digit_hist = (uint32_t*)(b + L.digit_hist);
    o.scan_status = (uint32_t*)(b + L.scan_status);
    o.counters = (uint32_t*)(b + L.counters);
    o.lookback = (uint32_t*)(b + L.lookback);
    o.zero_begin = b + L.zero_begin;
    o.zero_bytes = L.zero_end - L.zero_begin;
    o.racc = (double*)(b + L.racc);
    o.passes = L.passes;
    o.bits_per_pass = L.bits;
    o.key_bits = L.key_bits;
    o.radix_tiles = L.radix_tiles;
    o.scan_tiles = L.scan_tiles;
    return PIC_OK;
}

template <typename T, int D>
static int sort_keys_perm(const pic_grid_t& g, const pic_particles_t& in, int32_t* perm, int32_t* cell_offsets,
                          const SortWs& ws, cudaStream_t st)
{
    const int64_t n = in.n;
    const int C = (int)cells_of(g);
    mark_phase(PIC_PHASE_BEGIN, st);
    PIC_CUDA_OK(cudaMemsetAsync(ws.zero_begin, 0, ws.zero_bytes, st));
    if (n > 0) {
        int blocks = (int)std::min<int64_t>((n + 255) / 256, 148 * 8);
        k_keys_hist<T, D><<<blocks, 256, 0, st>>>(make_partp<T>(in), make_gridp<T>(g), n, ws.keys[0], ws.cell_count);
        count_launch();
    }
    mark_phase(PIC_PHASE_KEYS, st);
    k_scan_cells<<<(unsigned)ws.scan_tiles, kScanThreads, 0, st>>>(ws.cell_count, cell_offsets, C, ws.scan_status,
                                                                    ws.counters + 0, ws.digit_hist, ws.passes,
                                                                    ws.bits_per_pass);
    count_launch();
    if (n > 0) {
        k_scan_digits<<<ws.passes, kRadix, 0, st>>>(ws.digit_hist);
        count_launch();
        mark_phase(PIC_PHASE_SCAN, st);
        int src = 0;
        for (int q = 0; q < ws.passes; ++q) {
            const bool last = q == ws.passes - 1;
            const uint32_t* kin = ws.keys[src];
            const uint32_t* iin = q == 0 ? nullptr : ws.idx[src];
            uint32_t* kout = last ? nullptr : ws.keys[src ^ 1];
            uint32_t* iout = last ? (uint32_t*)perm : ws.idx[src ^ 1];
            k_radix_pass<<<(unsigned)ws.radix_tiles, kRadixThreads, 0, st>>>(
                kin, iin, kout, iout, n, q * ws.bits_per_pass, (1u << ws.bits_per_pass) - 1u, ws.digit_hist + q * kRadix, ws.counters + 1 + q,
                ws.lookback + (size_t)q * (size_t)ws.radix_tiles * kRadix);
            count_launch();
            src ^= 1;
        }
    }
    mark_phase(PIC_PHASE_RADIX, st);
    return cudaGetLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

template <typename T, int D>
static int sort_impl(const pic_grid_t& g, const pic_particles_t& in, pic_particles_t& out, int32_t* perm,
                     int32_t* cell_offsets, const SortWs& ws, bool reorder, cudaStream_t st)
{
    int rc = sort_keys_perm<T, D>(g, in, perm, cell_offsets, ws, st);
    if (rc != PIC_OK) return rc;
    const int64_t n = in.n;
    if (n > 0 && reorder) {
        k_reorder<T, D><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(make_partp<T>(in), make_partp<T>(out), perm, n);
        count_launch();
    }
    mark_phase(PIC_PHASE_REORDER, st);
    return cudaGetLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

int launch_sort(const pic_grid_t& g, const pic_particles_t& in, pic_particles_t& out, int32_t* perm,
                int32_t* cell_offsets, const SortWs& ws, bool reorder, cudaStream_t st)
{
    if (g.dtype == PIC_F32) {
        return g.dim == 2 ? sort_impl<float, 2>(g, in, out, perm, cell_offsets, ws, reorder, st)
                          : sort_impl<float, 3>(g, in, out, perm, cell_offsets, ws, reorder, st);
    }
    return g.dim == 2 ? sort_impl<double, 2>(g, in, out, perm, cell_offsets, ws, reorder, st)
                      : sort_impl<double, 3>(g, in, out, perm, cell_offsets, ws, reorder, st);
}

}  // namespace pic
