// pic_sort.cu -- stable counting sort of the particles by cell key (rows a1-a4 of the hot path).
//
// The paper sorts with histogram -> prefix sum -> atomic-counter scatter (section 3.2,
// Alg. 2 lines 1-5 PAPER.md:207-212), notes that hand-written CUDA histogram and prefix-sum
// kernels were worth a factor 2, and prefers, "for the rest of this paper", a
// sort for PRE-ORDERED particles that only moves the particles whose bucket changed (Alg. 2,
// PAPER.md:124, 190-196, 207-258; 23 % of the particles per step).  The atomic scatter
// is not stable; this build needs the unique stable permutation (R7).  It gets it from the same
// two ideas:
//
//   * cell_offsets as found ON ENTRY is read as a hint: intervals I_k = [hint[k], hint[k+1]) that
//     described the order of `in` at some earlier time (the previous step's output).  A particle
//     at position i is a STAYER if i lies in the interval of its NEW key, else a MOVER.  For any
//     non-decreasing hint the stable order of cell k is: movers into k from positions below I_k
//     (ascending position), the stayers of k (ascending position), movers from above I_k.  So only
//     the movers are sorted: they are compacted in position order (decoupled look-back) and go
//     through an LSD radix sort of (key, position) pairs, each pass a one-sweep stable partition
//     (warp-aggregated ranking, per-tile digit counts chained by decoupled look-back).  A hint that
//     is not non-decreasing within [0, N] (first call, garbage) makes every particle a mover: the
//     result is the same permutation, only slower.
//   * the full-key histogram and its exclusive scan give cell_offsets; the movers' histogram and
//     its scan place each mover inside its cell.
//
// Kernels:  k_hint_hist      hint -> private copy, validity flag; is this call the next link of a chain?  The three
//                            histograms: zero, or in a chain formed from the step kernel's per-cell in/out counters
//           k_classify       x[d] -> key (cell or bucket), histograms, stayer/mover split, movers staged per 2048 positions
//                            (returns at once in a chain: the previous step kernel has emitted all of it)
//           k_scan_cells     count[C] -> exclusive offsets [C+1] (single pass, decoupled look-back)
//           k_movers_place   staged movers -> one list in position order
//           k_scan_digits    digit histograms -> exclusive global digit offsets
//           k_radix_pass     one stable partition of the movers by an (at most) 8-bit digit; the last pass writes
//                            the movers' entries of perm
//           k_cell_base      per cell: where its stayers start in perm
//           k_perm_stayers   perm of the stayers
//           k_reorder        out_a[j] = in_a[perm[j]] value by value (most particles stay where they are)
//           k_pack_rec/k_unpack_rec  the same through 32-byte records (most particles move: first sort)
#include <cmath>
#include <cstring>

#include "pic_common.cuh"

namespace pic {

static inline size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

// ----------------------------------------------------------------------------- tile shapes
constexpr int kRadixThreads = 256;
#ifndef PIC_RADIX_IPT
#define PIC_RADIX_IPT 16
#endif
constexpr int kRadixIPT = PIC_RADIX_IPT;
constexpr int kRadixTile = kRadixThreads * kRadixIPT;      // 4096 pairs per tile
constexpr int kRadixWarps = kRadixThreads / 32;

constexpr int kScanThreads = 256;
constexpr int kScanIPT = 8;
constexpr int kScanTile = kScanThreads * kScanIPT;         // 2048 counts per tile

constexpr int kClsThreads = 256;
#ifndef PIC_CLS_IPT
#define PIC_CLS_IPT 16
#endif
constexpr int kClsIPT = PIC_CLS_IPT;
constexpr int kClsTile = kClsThreads * kClsIPT;            // 4096 positions per tile
constexpr int kClsWarps = kClsThreads / 32;

constexpr uint32_t kFlagAgg = 1u << 30, kFlagPrefix = 2u << 30, kValMask = (1u << 30) - 1;

// slots of SortWs::counters
enum { kCtrScanA = 0, kCtrScanB = 1, kCtrCls = 2, kCtrRadix = 3 /* .. +kMaxPasses */, kCtrMovers = 8, kCtrHintBad = 9, kCtrGate = 16, kCtrStrays = 17, kCtrChain = 18 };

__device__ __forceinline__ uint32_t ld_volatile(const uint32_t* p)
{
    return *reinterpret_cast<const volatile uint32_t*>(p);
}
__device__ __forceinline__ void st_volatile(uint32_t* p, uint32_t v)
{
    *reinterpret_cast<volatile uint32_t*>(p) = v;
}

// look-back of a single-value chain by one warp: returns the exclusive prefix of `tile`
__device__ __forceinline__ uint32_t warp_lookback(uint32_t* status, int tile, uint32_t total, unsigned lane)
{
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
    if (lane == 0 && tile != 0) st_volatile(&status[tile], kFlagPrefix | (excl + total));
    return excl;
}

// ----------------------------------------------------------------------------- the hint
// Is this call the next link of a chain (PIC_SORT_CHAINED, pic.h)?  Only if the caller asks for it AND the
// workspace holds the emission of a step that wrote exactly the arrays this call reads.
__device__ __forceinline__ bool chain_holds(const ChainSig* sig, const ChainSig& want)
{
    bool ok = sig->magic == kChainMagic && sig->n == want.n && sig->cells == want.cells && sig->grid == want.grid;
#pragma unroll
    for (int a = 0; a < 7; ++a) ok = ok && sig->arr[a] == want.arr[a];
    return ok;
}

// private copy of the hint: cell_offsets as found on entry, or -- in a chain -- the offsets the previous step
// wrote (kept in the workspace, so that the emitted stayer/mover split and the hint cannot disagree);
// bad = 1 unless 0 <= h[0] <= h[1] <= ... <= h[C] <= N.
// The same threads prepare the three histograms (one launch instead of three: small problems are launch bound).  Not a
// chain: they are zero before k_classify fills them.  A chain: they come from what the previous step kernel counted --
// particles that left each cell, movers into it, and how many of those come from below: count = old count - out + in.
// Every block decides "chain or not" for itself from the signature, so there is no dependence between blocks.
__global__ void __launch_bounds__(256) k_hint_hist(const int32_t* __restrict__ hint, const int32_t* __restrict__ prev_off,
                                                   const ChainSig* __restrict__ sig, ChainSig want, int chain_req,
                                                   int32_t* __restrict__ old_off, int C, int64_t n, uint32_t* counters,
                                                   const int32_t* __restrict__ cell_out, const unsigned long long* __restrict__ mover_in,
                                                   int32_t* __restrict__ cell_count, int32_t* __restrict__ mover_count,
                                                   int32_t* __restrict__ mover_lo)
{
    __shared__ int s_chain;
    if (threadIdx.x == 0) {
        s_chain = (chain_req && chain_holds(sig, want)) ? 1 : 0;
        if (blockIdx.x == 0) counters[kCtrChain] = (uint32_t)s_chain;
    }
    __syncthreads();
    const int32_t* __restrict__ h = s_chain ? prev_off : hint;
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k > C) return;
    const int32_t a = h[k];
    old_off[k] = a;
    bool bad = a < 0 || (int64_t)a > n;
    int32_t b = a;
    if (k < C) {
        b = h[k + 1];
        bad = bad || b < a;
    }
    if (bad) counters[kCtrHintBad] = 1u;
    if (!s_chain) {
        cell_count[k] = 0;
        mover_count[k] = 0;
        mover_lo[k] = 0;
    } else if (k < C) {
        const unsigned long long in = mover_in[k];
        const int32_t min = (int32_t)(uint32_t)in;
        mover_count[k] = min;
        mover_lo[k] = (int32_t)(uint32_t)(in >> 32);
        cell_count[k] = b - a - cell_out[k] + min;
    }
}

// the step has left its emission behind: the next call may chain on to it
__global__ void k_chain_commit(ChainSig* sig, ChainSig now) { *sig = now; }

// ----------------------------------------------------------------------------- keys, histograms, stayer/mover split
// a1: key = c_x + n_x*(c_y + n_y*c_z) (x fastest), clamped cell index
// (PAPER.md:493-497).  a2: count[key]++ -- consecutive lanes holding the same key (the common
// case once the particles are pre-ordered) are merged into one atomic per run.
// Movers (see the header) are appended to (mkey, midx) in position order; mask / mprefix hold,
// per 32 positions, the movers' bits and the number of movers before the word.
// Per-block hash table key -> (count, movers, movers from below) in shared memory (open addressing, 8 probes;
// a key that finds no slot goes straight to the global histograms).  Counts of a block are at most
// kClsTile = 2^12: count and movers share one word (13 bits each).
constexpr int kHashBits = 10, kHashSize = 1 << kHashBits;
struct BlockHist {
    uint32_t* key;      // [kHashSize], 0xFFFFFFFF = empty
    uint32_t* c01;      // [kHashSize] count | movers << 13
    uint32_t* c2;       // [kHashSize] movers from below
    int32_t *cell_count, *mover_count, *mover_lo;
    __device__ __forceinline__ void add(uint32_t k, uint32_t c0, uint32_t c1, uint32_t cl) const
    {
        uint32_t slot = (k * 2654435761u) >> (32 - kHashBits);
#pragma unroll 1
        for (int probe = 0; probe < 8; ++probe) {
            const uint32_t old = atomicCAS(&key[slot], 0xFFFFFFFFu, k);
            if (old == 0xFFFFFFFFu || old == k) {
                atomicAdd(&c01[slot], c0 | (c1 << 13));
                if (cl) atomicAdd(&c2[slot], cl);
                return;
            }
            slot = (slot + 1) & (kHashSize - 1);
        }
        atomicAdd(&cell_count[k], (int)c0);
        if (c1) atomicAdd(&mover_count[k], (int)c1);
        if (cl) atomicAdd(&mover_lo[k], (int)cl);
    }
};
static_assert(kClsTile <= (1 << 12), "13-bit fields of BlockHist");
static_assert(kClsTile % kStageTile == 0 && kStageTile % (32 * kClsIPT) == 0, "staging tiles are whole warps of a classify block");

// One warp's 32*kClsIPT positions.  CHECK = false: all of them are below n (no bounds tests).
template <typename T, int D, bool CHECK, bool BK>
__device__ __forceinline__ void classify_warp(const PartP<T>& p, const GridP<T>& g, int n, int wbase, unsigned lane, bool hint_ok,
                                              const int32_t* __restrict__ old_off, const BlockHist& hist,
                                              uint32_t* __restrict__ pkey, uint32_t (&key)[kClsIPT], uint32_t (&bal)[kClsIPT],
                                              uint32_t& mover_bits, uint32_t& lo_bits)
{
    const int i0 = wbase + (int)lane;
    // all positions of this thread first: independent loads
    T xs[D][kClsIPT];
#pragma unroll
    for (int c = 0; c < D; ++c) {
        const T* __restrict__ xc = p.x[c] + i0;
#pragma unroll
        for (int r = 0; r < kClsIPT; ++r) xs[c][r] = (!CHECK || i0 + r * 32 < n) ? xc[r * 32] : (T)0;
    }
#pragma unroll
    for (int r = 0; r < kClsIPT; ++r) {
        int cell[3] = {0, 0, 0};
#pragma unroll
        for (int c = 0; c < D; ++c) cell[c] = cell_index(grid_coord(xs[c][r], g.h[c], g.inv_h[c], g.hmul), g.n[c]);
        const int k = sort_key<T, D, BK>(g, cell);
        key[r] = (!CHECK || i0 + r * 32 < n) ? (uint32_t)k : 0xFFFFFFFFu;
        if (!CHECK || i0 + r * 32 < n) pkey[i0 + r * 32] = (uint32_t)k;
    }
    // the hint intervals of the new keys: independent loads again.  stayer <=> ha <= i < hb
    mover_bits = 0;
    lo_bits = 0;
    if (hint_ok) {
        int32_t ha[kClsIPT], hb[kClsIPT];
#pragma unroll
        for (int r = 0; r < kClsIPT; ++r) {
            const bool valid = !CHECK || key[r] != 0xFFFFFFFFu;
            ha[r] = valid ? old_off[key[r]] : 0;
            hb[r] = valid ? old_off[key[r] + 1] : 0;
        }
#pragma unroll
        for (int r = 0; r < kClsIPT; ++r) {
            const int i = i0 + r * 32;
            const bool valid = !CHECK || key[r] != 0xFFFFFFFFu;
            const bool stay = (unsigned)(i - ha[r]) < (unsigned)(hb[r] - ha[r]);     // ha <= hb: the hint is non-decreasing
            if (valid && !stay) mover_bits |= 1u << r;
            if (valid && i < ha[r]) lo_bits |= 1u << r;
        }
    } else {
#pragma unroll
        for (int r = 0; r < kClsIPT; ++r)
            if (!CHECK || key[r] != 0xFFFFFFFFu) mover_bits |= 1u << r;
    }
    // the three histograms (all keys, movers, movers from below): one entry per run of equal keys in a
    // row of 32 positions (the common case once the particles are pre-ordered) goes to the
    // block's hash table in shared memory; the table is flushed with one global atomic per key and
    // histogram, so the number of global atomics on one address does not grow with the density (clustered
    // config 4: same-address atomics serialise in L2 and made this kernel 3.7x slower)
    // (dense = the warp's 512 positions span at most three cells; elsewhere the addresses are spread and the
    // atomics go straight to the grid arrays, which is cheaper than hashing)
    const uint32_t kfirst = __shfl_sync(0xFFFFFFFFu, key[0], 0), klast = __shfl_sync(0xFFFFFFFFu, key[kClsIPT - 1], 31);
    const bool dense = klast - kfirst <= 2u;
#pragma unroll
    for (int r = 0; r < kClsIPT; ++r) {
        bal[r] = __ballot_sync(0xFFFFFFFFu, (mover_bits >> r) & 1u);
        const unsigned lob = __ballot_sync(0xFFFFFFFFu, (lo_bits >> r) & 1u);
        const uint32_t prev = __shfl_up_sync(0xFFFFFFFFu, key[r], 1);
        const bool head = (lane == 0) || (prev != key[r]);
        const unsigned heads = __ballot_sync(0xFFFFFFFFu, head);
        if (head && (!CHECK || key[r] != 0xFFFFFFFFu)) {
            const unsigned above = heads & ~((2u << lane) - 1);      // heads strictly above this lane
            const int next = above ? __ffs(above) - 1 : 32;
            // a run never extends over the invalid lanes of a ragged last word: those carry key
            // 0xFFFFFFFF, so the first of them is a head
            const unsigned run = (next == 32 ? 0xFFFFFFFFu : ((1u << next) - 1u)) & ~((1u << lane) - 1u);
            const uint32_t c0 = (uint32_t)(next - (int)lane), c1 = (uint32_t)__popc(bal[r] & run), cl = (uint32_t)__popc(lob & run);
            if (dense) {
                hist.add(key[r], c0, c1, cl);
            } else {
                atomicAdd(&hist.cell_count[key[r]], (int)c0);
                if (c1) atomicAdd(&hist.mover_count[key[r]], (int)c1);
                if (cl) atomicAdd(&hist.mover_lo[key[r]], (int)cl);
            }
        }
    }
}

template <typename T, int D, bool BK>
#ifndef PIC_CLS_MINB
#define PIC_CLS_MINB 4
#endif
__global__ void __launch_bounds__(kClsThreads, (sizeof(T) == 8 ? PIC_CLS_MINB / 2 : PIC_CLS_MINB))   // (doubles: 64 registers spill)
k_classify(PartP<T> p, GridP<T> g, int n, const int32_t* __restrict__ old_off, int32_t* __restrict__ cell_count,
           int32_t* __restrict__ mover_count, int32_t* __restrict__ mover_lo, uint32_t* __restrict__ mkey,
           uint32_t* __restrict__ midx, uint32_t* __restrict__ mask, uint32_t* __restrict__ mprefix,
           int32_t* __restrict__ tile_count, uint32_t* __restrict__ pkey, const uint32_t* __restrict__ counters)
{
    __shared__ uint32_t s_wsum[kClsWarps];
    if (counters[kCtrChain]) return;                  // a chain: the previous step kernel has done this work
    const unsigned tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = (int)blockIdx.x;
    const bool hint_ok = counters[kCtrHintBad] == 0u;
    const int wbase = tile * kClsTile + (int)warp * (32 * kClsIPT);

    __shared__ uint32_t s_hkey[kHashSize], s_hc01[kHashSize], s_hc2[kHashSize];
    for (int q = tid; q < kHashSize; q += kClsThreads) { s_hkey[q] = 0xFFFFFFFFu; s_hc01[q] = 0u; s_hc2[q] = 0u; }
    __syncthreads();
    const BlockHist hist{s_hkey, s_hc01, s_hc2, cell_count, mover_count, mover_lo};

    uint32_t key[kClsIPT], bal[kClsIPT];
    uint32_t mover_bits, lo_bits;
    if (wbase + 32 * kClsIPT <= n)
        classify_warp<T, D, false, BK>(p, g, n, wbase, lane, hint_ok, old_off, hist, pkey, key, bal, mover_bits, lo_bits);
    else
        classify_warp<T, D, true, BK>(p, g, n, wbase, lane, hint_ok, old_off, hist, pkey, key, bal, mover_bits, lo_bits);

    // movers before each word of this warp, warp total
    uint32_t wpre[kClsIPT], wtotal = 0;
#pragma unroll
    for (int r = 0; r < kClsIPT; ++r) { wpre[r] = wtotal; wtotal += __popc(bal[r]); }
    if (lane == 0) s_wsum[warp] = wtotal;
    __syncthreads();
    // movers are staged per kStageTile positions (one warp's range in the step kernel, which writes the same
    // layout when it emits): this block covers kClsTile / kStageTile of them
    constexpr int kWarpsPerStage = kStageTile / (32 * kClsIPT);
    const int half = (int)warp / kWarpsPerStage;
    uint32_t warp_off = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kClsWarps; ++w) {
        const uint32_t t = s_wsum[w];
        if (w / kWarpsPerStage == half) {
            if (w < (int)warp) warp_off += t;
            total += t;
        }
    }
    if ((int)tid % (32 * kWarpsPerStage) == 0 && (int64_t)(tile * (kClsTile / kStageTile) + half) * kStageTile < n)
        tile_count[tile * (kClsTile / kStageTile) + half] = (int32_t)total;
    // the block's histograms go to the grid arrays: one atomic per key and histogram (after the barrier above)
    for (int q = tid; q < kHashSize; q += kClsThreads) {
        const uint32_t k = s_hkey[q];
        if (k != 0xFFFFFFFFu) {
            const uint32_t v = s_hc01[q], l = s_hc2[q];
            atomicAdd(&cell_count[k], (int)(v & 0x1FFFu));
            if (v >> 13) atomicAdd(&mover_count[k], (int)(v >> 13));
            if (l) atomicAdd(&mover_lo[k], (int)l);
        }
    }
    // tile-relative for now: k_movers_place adds the movers of the tiles before this one
    const uint32_t base = warp_off;
    const int stage = tile * kClsTile + half * kStageTile;
    const unsigned lt = (1u << lane) - 1;
    // lane r writes the mask and prefix words of row r (the ballots are the same in every lane)
    {
        uint32_t my_bal = 0, my_pre = 0;
#pragma unroll
        for (int r = 0; r < kClsIPT; ++r)
            if ((int)lane == r) { my_bal = bal[r]; my_pre = wpre[r]; }
        const int iw = wbase + (int)lane * 32;
        if (lane < kClsIPT && iw < n) {
            mask[iw >> 5] = my_bal;
            mprefix[iw >> 5] = base + my_pre;
        }
    }
#pragma unroll
    for (int r = 0; r < kClsIPT; ++r) {
        if ((mover_bits >> r) & 1u) {
            const int dst = stage + (int)(base + wpre[r]) + __popc(bal[r] & lt);
            mkey[dst] = key[r];
            midx[dst] = (uint32_t)(wbase + r * 32 + (int)lane);
        }
    }
}

// The movers of staging tile t (written by k_classify, or by the previous step kernel in a chain) move from
// [t*kStageTile, ...) to their place in the global list: tile_base[t] = number of movers in the tiles before t
// (exclusive scan of tile_count).  The per-word mover prefixes become global too.
__global__ void __launch_bounds__(256)
k_movers_place(const uint32_t* __restrict__ stage_key, const uint32_t* __restrict__ stage_idx, uint32_t* __restrict__ mkey,
               uint32_t* __restrict__ midx, uint32_t* __restrict__ mask, uint32_t* __restrict__ mprefix,
               const int32_t* __restrict__ tile_base, int ntiles, int64_t n, uint32_t* counters, ChainSig* sig)
{
    const int tile = (int)blockIdx.x, tid = threadIdx.x;
    const uint32_t base = (uint32_t)tile_base[tile];
    const int cnt = tile_base[tile + 1] - tile_base[tile];
    const int64_t stage = (int64_t)tile * kStageTile;
    for (int r = tid; r < cnt; r += 256) {
        mkey[base + r] = stage_key[stage + r];
        midx[base + r] = stage_idx[stage + r];
    }
    const int64_t w0 = stage >> 5, nwords = (n + 31) / 32;
    for (int w = tid; w < kStageTile / 32 && w0 + w < nwords; w += 256) mprefix[w0 + w] += base;
    if (tile == ntiles - 1 && tid == 0) {                // total number of movers, sentinel word
        const uint32_t total = (uint32_t)tile_base[ntiles];
        counters[kCtrMovers] = total;
        counters[kCtrGate] = (2 * (int64_t)total > n) ? 1u : 0u;      // most particles move: reorder before the step kernel
        mask[nwords] = 0u;
        mprefix[nwords] = total;
        sig->magic = 0;                                  // the emission is used up (the step kernel writes the next one)
    }
}

// ----------------------------------------------------------------------------- exclusive scan of per-cell counts
// a3: offsets[k] = sum_{k'<k} count[k'], offsets[C] = total ("prefix sum").
// Single pass: each tile publishes its aggregate, then looks back over its predecessors.
// With digit_hist != NULL the per-pass digit histograms of the radix sort are summed here from
// the counts (C cells instead of one pass over the keys).
__global__ void __launch_bounds__(kScanThreads) k_scan_cells(const int32_t* __restrict__ count, int32_t* __restrict__ offsets,
                                                              int C, uint32_t* status, uint32_t* tile_counter,
                                                              uint32_t* __restrict__ digit_hist, int passes, int bits,
                                                              int32_t* __restrict__ offsets2 = nullptr)
{
    __shared__ uint32_t s_warp[kScanThreads / 32];
    __shared__ uint32_t s_tile, s_excl;
    __shared__ uint32_t s_hist[kMaxPasses][kRadix];
    if (threadIdx.x == 0) s_tile = atomicAdd(tile_counter, 1u);
    if (digit_hist)
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
    if (digit_hist) {
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

    if (warp == 0) {
        const uint32_t excl = warp_lookback(status, tile, total, lane);
        if (lane == 0) s_excl = excl;
    }
    __syncthreads();
    uint32_t run = s_excl + excl_thread;
#pragma unroll
    for (int k = 0; k < kScanIPT; ++k) {
        if (base + k < C) {
            offsets[base + k] = (int32_t)run;
            if (offsets2) offsets2[base + k] = (int32_t)run;
        }
        run += v[k];
        if (base + k == C - 1) {
            offsets[C] = (int32_t)run;
            if (offsets2) offsets2[C] = (int32_t)run;
        }
    }
    if (digit_hist) {
        for (int i = threadIdx.x; i < passes * kRadix; i += kScanThreads) {
            uint32_t c = (&s_hist[0][0])[i];
            if (c) atomicAdd(&digit_hist[i], c);
        }
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

// zero the look-back words the radix passes will use: passes x tiles(number of movers) x kRadix
__global__ void __launch_bounds__(256) k_zero_lookback(uint32_t* lookback, const uint32_t* __restrict__ counters, int passes,
                                                       int64_t pass_stride)
{
    const int64_t tiles = ((int64_t)counters[kCtrMovers] + kRadixTile - 1) / kRadixTile;
    const int64_t words = tiles * kRadix;
    for (int q = 0; q < passes; ++q)
        for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < words; i += (int64_t)gridDim.x * blockDim.x)
            lookback[q * pass_stride + i] = 0u;
}

// ----------------------------------------------------------------------------- one radix pass over the movers
// Stable partition of (key, idx) pairs by digit (key >> shift) & mask (at most 8 bits).  Tile-local order is
// (warp, round, lane) = ascending input position, so equal digits keep their input order.
// keys_out == nullptr: keys are not needed any more (last pass).  The number of pairs is read
// from the device (counters[kCtrMovers]); blocks beyond the last tile exit at once.
#ifndef PIC_RADIX_MINB
#define PIC_RADIX_MINB 5        // resident blocks per SM k_radix_pass is compiled for (48 registers)
#endif
// LAST: the pairs leave this pass sorted by (key, position), so the place of each in perm is known here and the
// sorted list is never written: the r-th mover of key k goes below the stayers of k if it comes from below the
// hint interval of k, else above them.
struct PermP {
    const int32_t* new_off;      // [C+1] cell_offsets of this sort
    const int32_t* mover_off;    // [C+1] exclusive scan of the movers' histogram
    const int32_t* old_off;      // [C+1] the hint
    int32_t* perm;
};
template <bool LAST>
__global__ void __launch_bounds__(kRadixThreads, PIC_RADIX_MINB)
k_radix_pass(const uint32_t* __restrict__ keys_in, const uint32_t* __restrict__ idx_in,
             uint32_t* __restrict__ keys_out, uint32_t* __restrict__ idx_out, const uint32_t* __restrict__ counters,
             int shift, uint32_t mask, const uint32_t* __restrict__ digit_offsets, uint32_t* tile_counter,
             uint32_t* lookback, PermP pp)
{
    __shared__ uint32_t s_cnt[kRadixWarps][kRadix];   // per-warp digit counters -> per-warp bases
    __shared__ uint32_t s_start[kRadix];              // tile-local start of each digit
    __shared__ uint32_t s_base[kRadix];               // global address of local position 0 of each digit
    __shared__ uint32_t s_keys[kRadixTile];
    __shared__ uint32_t s_idx[kRadixTile];
    __shared__ uint32_t s_wsum[kRadixWarps];
    __shared__ uint32_t s_tile;

    const int64_t n = counters[kCtrMovers];
    if ((int64_t)blockIdx.x * kRadixTile >= n) return;   // as many blocks run as there are tiles
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
        val[r] = ok ? idx_in[tile_base + loc] : 0u;
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
    const bool hint_ok = counters[kCtrHintBad] == 0u;
    for (int q = tid; q < tile_valid; q += kRadixThreads) {
        uint32_t k = s_keys[q];
        uint32_t dst = s_base[(k >> shift) & mask] + q;
        if constexpr (LAST) {
            const int32_t i = (int32_t)s_idx[q];
            const int32_t m0 = pp.mover_off[k], m1 = pp.mover_off[k + 1];
            const int32_t n0 = pp.new_off[k], n1 = pp.new_off[k + 1];
            const int32_t stay = (n1 - n0) - (m1 - m0);
            const bool below = hint_ok && i < pp.old_off[k];
            pp.perm[n0 + ((int32_t)dst - m0) + (below ? 0 : stay)] = i;
        } else {
            keys_out[dst] = k;
            idx_out[dst] = s_idx[q];
        }
    }
}

// ----------------------------------------------------------------------------- perm
// cell_base[k] = new_off[k] + (#movers into k from below) - a_k + (#movers before position a_k),
// so that the stayer at position i of cell k goes to cell_base[k] + i - (#movers before i).
__global__ void __launch_bounds__(256) k_cell_base(const int32_t* __restrict__ new_off, const int32_t* __restrict__ old_off,
                                                   const int32_t* __restrict__ mover_lo, const uint32_t* __restrict__ mask,
                                                   const uint32_t* __restrict__ mprefix, int32_t* __restrict__ cell_base, int C,
                                                   const uint32_t* __restrict__ counters)
{
    if (counters[kCtrHintBad]) return;                 // no stayers
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= C) return;
    const int32_t a = old_off[k];
    const uint32_t mv = mprefix[a >> 5] + __popc(mask[a >> 5] & ((1u << (a & 31)) - 1u));
    cell_base[k] = new_off[k] + mover_lo[k] - a + (int32_t)mv;
}

// stayers: position i (mover bit clear) kept its cell k = pkey[i] and goes to
// cell_base[k] + i - (#movers before i).  Coalesced over positions; the mask word is one broadcast load.
#ifndef PIC_STAY_IPT
#define PIC_STAY_IPT 4
#endif
constexpr int kStayIPT = PIC_STAY_IPT;
__global__ void __launch_bounds__(256)
k_perm_stayers(const uint32_t* __restrict__ pkey, const int32_t* __restrict__ cell_base, const uint32_t* __restrict__ mask,
               const uint32_t* __restrict__ mprefix, int32_t* __restrict__ perm, int n, const uint32_t* __restrict__ counters)
{
    if (counters[kCtrHintBad]) return;                 // no stayers
    const int base = ((int)blockIdx.x * 256 + (int)(threadIdx.x & ~31u)) * kStayIPT + (int)(threadIdx.x & 31u);
    uint32_t m[kStayIPT], pre[kStayIPT], k[kStayIPT];
#pragma unroll
    for (int r = 0; r < kStayIPT; ++r) {
        const int i = base + r * 32;
        m[r] = i < n ? mask[i >> 5] : 0xFFFFFFFFu;
        pre[r] = i < n ? mprefix[i >> 5] : 0u;
        k[r] = i < n ? pkey[i] : 0u;
    }
    const uint32_t bit = 1u << (threadIdx.x & 31u);
#pragma unroll
    for (int r = 0; r < kStayIPT; ++r) {
        const int i = base + r * 32;
        if (!(m[r] & bit)) {
            const int mv = (int)(pre[r] + __popc(m[r] & (bit - 1u)));
            perm[cell_base[k[r]] + i - mv] = i;
        }
    }
}

// ----------------------------------------------------------------------------- reorder
// a4: out_a[j] = in_a[perm[j]] for all attributes, bit for bit; coalesced writes, gathered reads.
template <typename T, int D>
__global__ void __launch_bounds__(256) k_reorder(PartP<T> in, PartP<T> out, const int32_t* __restrict__ perm, int64_t n,
                                                 const uint32_t* __restrict__ gate, uint32_t want)
{
    if (gate && *gate != want) return;
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = perm[j];
        T x[D], v[D];
#pragma unroll
        for (int c = 0; c < D; ++c) { x[c] = in.x[c][i]; v[c] = in.v[c][i]; }
        const T w = in.w[i];
#pragma unroll
        for (int c = 0; c < D; ++c) { out.x[c][j] = x[c]; out.v[c][j] = v[c]; }
        out.w[j] = w;
    }
}

// The same reorder when perm is (nearly) random -- the first sort of particles in random order.  k_reorder then
// fetches one 32-byte sector per 4- or 8-byte value: A sectors per particle (16.4 ms for 1e8 fp32 particles, 3-D).
// Here a whole sector of attributes travels together: K = 32/sizeof(T) attribute arrays are interleaved into 32-byte
// records (coalesced both ways), then slot j fetches record perm[j] with ONE scattered sector and writes its K
// attributes (coalesced).  ceil(A/K) rounds (one in fp32, two in fp64) through a 32 N byte scratch (the movers'
// key/index arrays and the per-position keys, free once perm exists, plus 12 N bytes of their own).  "Scattered ... a
// multiple of 32 bytes for every moved particle" is the paper's cost of moving a particle: this keeps
// it at one such access per particle (fp32) instead of one per value.
template <typename T>
struct RecPtrs {
    const T* s[8];
    T* d[8];
};

template <typename T>
__global__ void __launch_bounds__(256) k_pack_rec(RecPtrs<T> a, uint4* __restrict__ rec, int64_t n,
                                                  const uint32_t* __restrict__ gate, uint32_t want)
{
    if (gate && *gate != want) return;
    constexpr int K = 32 / (int)sizeof(T);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        union { uint4 q[2]; T v[K]; } r;
        r.q[0] = make_uint4(0u, 0u, 0u, 0u);
        r.q[1] = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
        for (int k = 0; k < K; ++k)
            if (a.s[k]) r.v[k] = a.s[k][i];
        rec[2 * i] = r.q[0];
        rec[2 * i + 1] = r.q[1];
    }
}

template <typename T>
__global__ void __launch_bounds__(256) k_unpack_rec(RecPtrs<T> a, const uint4* __restrict__ rec, const int32_t* __restrict__ perm,
                                                    int64_t n, const uint32_t* __restrict__ gate, uint32_t want)
{
    if (gate && *gate != want) return;
    constexpr int K = 32 / (int)sizeof(T);
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < n; j += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = perm[j];
        union { uint4 q[2]; T v[K]; } r;
        r.q[0] = __ldg(rec + 2 * i);
        r.q[1] = __ldg(rec + 2 * i + 1);
#pragma unroll
        for (int k = 0; k < K; ++k)
            if (a.d[k]) a.d[k][j] = r.v[k];
    }
}

template <typename T>
static int reorder_records(const pic_grid_t& g, const pic_particles_t& in, const pic_particles_t& out, const int32_t* perm,
                           void* scratch, const uint32_t* gate, uint32_t want, cudaStream_t st)
{
    const int64_t n = in.n;
    constexpr int K = 32 / (int)sizeof(T);
    const T* src[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    T* dst[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    int A = 0;
    for (int c = 0; c < g.dim; ++c) { src[A] = (const T*)in.x[c]; dst[A++] = (T*)out.x[c]; }
    src[A] = (const T*)in.w; dst[A++] = (T*)out.w;              // positions and weight together, then the velocities
    for (int c = 0; c < g.dim; ++c) { src[A] = (const T*)in.v[c]; dst[A++] = (T*)out.v[c]; }
    const int64_t want_blocks = (n + 255) / 256, cap = (int64_t)sm_count() * 8;
    const unsigned blocks = (unsigned)(want_blocks < cap ? want_blocks : cap);
    for (int a = 0; a < A; a += K) {
        RecPtrs<T> rp;
        for (int k = 0; k < 8; ++k) {
            const bool on = k < K && a + k < A;
            rp.s[k] = on ? src[a + k] : nullptr;
            rp.d[k] = on ? dst[a + k] : nullptr;
        }
        k_pack_rec<T><<<blocks, 256, 0, st>>>(rp, (uint4*)scratch, n, gate, want);
        k_unpack_rec<T><<<blocks, 256, 0, st>>>(rp, (const uint4*)scratch, perm, n, gate, want);
        count_launch(2);
    }
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

// out_a[j] = in_a[perm[j]] when *gate == want, through 32-byte records (see k_pack_rec); scratch: 32 N bytes
int launch_reorder_records(const pic_grid_t& g, const pic_particles_t& in, const pic_particles_t& out, const int32_t* perm,
                           void* scratch, const uint32_t* gate, uint32_t want, cudaStream_t st)
{
    if (in.n <= 0) return PIC_OK;
    return g.dtype == PIC_F32 ? reorder_records<float>(g, in, out, perm, scratch, gate, want, st)
                              : reorder_records<double>(g, in, out, perm, scratch, gate, want, st);
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
    size_t keys0, keys1, idx0, idx1, pkey, rec_extra, mask, mprefix, old_off, prev_off, mover_off, cell_base, tile_count, tile_base, lookback;
    size_t hist_begin, cell_count, mover_count, mover_lo, hist_end, emit_begin, cell_out, mover_in, emit_end;
    size_t zero_begin, digit_hist, scan_status, cls_status, counters, zero_end;
    size_t chain_sig, racc, total;
    int passes, bits, key_bits;
    int64_t radix_tiles, scan_tiles, cls_tiles, stage_tiles;
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
    L.cls_tiles = (n + kClsTile - 1) / kClsTile;
    L.stage_tiles = (n + kStageTile - 1) / kStageTile;
    // The chain signature comes FIRST, at an offset that does not depend on n or the grid: whatever else is done with
    // this workspace -- a carve for another particle count, the field solve's arrays, a caller's own data -- lands on
    // it (or is one of this library's calls, which void it) before it can reach the emission the signature vouches for.
    size_t off = 0;
    L.chain_sig = off; off += 256;
    const size_t nb = align256(sizeof(uint32_t) * (size_t)(n > 0 ? n : 1));
    const size_t wb = align256(sizeof(uint32_t) * (size_t)((n + 31) / 32 + 2));
    const size_t cb = align256(sizeof(int32_t) * (size_t)(C + 1));
    L.keys0 = off; off += nb;
    L.keys1 = off; off += nb;
    L.idx0 = off; off += nb;
    L.idx1 = off; off += nb;
    L.pkey = off; off += nb;
    L.rec_extra = off; off += align256(12 * (size_t)(n > 0 ? n : 1));      // keys0 .. here: the 32 N byte record scratch
    L.mask = off; off += wb;
    L.mprefix = off; off += wb;
    L.old_off = off; off += cb;
    L.prev_off = off; off += cb;
    L.mover_off = off; off += cb;
    L.cell_base = off; off += cb;
    L.tile_count = off; off += align256(sizeof(int32_t) * (size_t)(L.stage_tiles + 1));
    L.tile_base = off; off += align256(sizeof(int32_t) * (size_t)(L.stage_tiles + 2));
    L.lookback = off; off += align256(sizeof(uint32_t) * (size_t)L.passes * (size_t)(L.radix_tiles > 0 ? L.radix_tiles : 1) * kRadix);
    L.hist_begin = off;
    L.cell_count = off; off += cb;
    L.mover_count = off; off += cb;
    L.mover_lo = off; off += cb;
    L.hist_end = off;
    L.emit_begin = off;
    L.cell_out = off; off += cb;
    L.mover_in = off; off += align256(sizeof(unsigned long long) * (size_t)(C + 1));
    L.emit_end = off;
    L.zero_begin = off;
    L.digit_hist = off; off += align256(sizeof(uint32_t) * kMaxPasses * kRadix);
    L.scan_status = off; off += align256(sizeof(uint32_t) * 2 * (size_t)L.scan_tiles);
    L.cls_status = off; off += align256(sizeof(uint32_t) * (size_t)((L.stage_tiles + kScanTile - 1) / kScanTile + 1));
    L.counters = off; off += 256;
    L.zero_end = off;
    L.racc = off; off += align256(sizeof(double) * (size_t)C);
    L.total = off;
    return L;
}

size_t sort_ws_bytes(const pic_grid_t& g, int64_t n) { return sort_layout(g, n).total; }

// number of sort keys: cells, or buckets of bucket[c] cells per dimension
int64_t sort_keys_of(const pic_grid_t& g, const int32_t* bucket)
{
    int64_t K = 1;
    for (int c = 0; c < g.dim; ++c) K *= bucket ? (g.n[c] + bucket[c] - 1) / bucket[c] : g.n[c];
    return K;
}

int carve_sort_ws(const pic_grid_t& g, int64_t n, void* ws, size_t ws_bytes, SortWs& o, const int32_t* bucket)
{
    SortLayout L = sort_layout(g, n);
    if (ws_bytes < L.total) return PIC_ERR_WORKSPACE;
    if (bucket) {                                        // fewer keys than cells: the arrays are large enough; fewer radix bits
        const int64_t K = sort_keys_of(g, bucket);
        int b = 1;
        while (((int64_t)1 << b) < K) ++b;
        L.key_bits = b;
        L.passes = (b + kRadixBits - 1) / kRadixBits;
        L.bits = (b + L.passes - 1) / L.passes;
        L.scan_tiles = (K + kScanTile - 1) / kScanTile;
    }
    o.nkeys = sort_keys_of(g, bucket);
    o.bucket = bucket;
    char* b = (char*)ws;
    o.keys[0] = (uint32_t*)(b + L.keys0);
    o.keys[1] = (uint32_t*)(b + L.keys1);
    o.idx[0] = (uint32_t*)(b + L.idx0);
    o.idx[1] = (uint32_t*)(b + L.idx1);
    o.mask = (uint32_t*)(b + L.mask);
    o.mprefix = (uint32_t*)(b + L.mprefix);
    o.old_off = (int32_t*)(b + L.old_off);
    o.prev_off = (int32_t*)(b + L.prev_off);
    o.chain_sig = (ChainSig*)(b + L.chain_sig);
    o.hist_begin = b + L.hist_begin;
    o.hist_bytes = L.hist_end - L.hist_begin;
    o.emit_begin = b + L.emit_begin;
    o.emit_bytes = L.emit_end - L.emit_begin;
    o.mover_off = (int32_t*)(b + L.mover_off);
    o.cell_base = (int32_t*)(b + L.cell_base);
    o.pkey = (uint32_t*)(b + L.pkey);
    o.tile_count = (int32_t*)(b + L.tile_count);
    o.tile_base = (int32_t*)(b + L.tile_base);
    o.lookback = (uint32_t*)(b + L.lookback);
    o.cell_count = (int32_t*)(b + L.cell_count);
    o.mover_count = (int32_t*)(b + L.mover_count);
    o.mover_lo = (int32_t*)(b + L.mover_lo);
    o.digit_hist = (uint32_t*)(b + L.digit_hist);
    o.scan_status = (uint32_t*)(b + L.scan_status);
    o.cls_status = (uint32_t*)(b + L.cls_status);
    o.counters = (uint32_t*)(b + L.counters);
    o.gate = o.counters + kCtrGate;
    o.stray_count = o.counters + kCtrStrays;
    o.stray_list = o.idx[0];
    o.rec_scratch = b + L.keys0;                         // keys0, keys1, idx0, idx1, pkey, rec_extra: 32 N bytes in a row
    o.zero_begin = b + L.zero_begin;
    o.zero_bytes = L.zero_end - L.zero_begin;
    o.racc = (double*)(b + L.racc);
    o.passes = L.passes;
    o.bits_per_pass = L.bits;
    o.key_bits = L.key_bits;
    o.radix_tiles = L.radix_tiles;
    o.scan_tiles = L.scan_tiles;
    o.cls_tiles = L.cls_tiles;
    o.stage_tiles = L.stage_tiles;
    o.emit = EmitP{o.pkey, o.mask, o.mprefix, o.keys[1], o.idx[1], o.tile_count, (int32_t*)(b + L.cell_out),
                   (unsigned long long*)(b + L.mover_in)};
    return PIC_OK;
}

// what identifies the particle set `p` on grid g (see ChainSig)
ChainSig chain_sig_of(const pic_grid_t& g, const pic_particles_t& p)
{
    ChainSig s;
    s.magic = kChainMagic;
    s.n = (uint64_t)p.n;
    s.cells = (uint64_t)cells_of(g);
    uint64_t h = 1469598103934665603ull;                 // FNV-1a over the grid parameters
    auto mix = [&](uint64_t v) { for (int k = 0; k < 8; ++k) { h ^= (v >> (8 * k)) & 0xFFu; h *= 1099511628211ull; } };
    mix((uint64_t)g.dim); mix((uint64_t)g.order); mix((uint64_t)g.dtype);
    for (int c = 0; c < g.dim; ++c) {
        uint64_t hb;
        memcpy(&hb, &g.h[c], 8);
        mix((uint64_t)g.n[c]); mix(hb);
    }
    s.grid = h;
    for (int c = 0; c < 3; ++c) {
        s.arr[c] = c < g.dim ? (uint64_t)(uintptr_t)p.x[c] : 0;
        s.arr[3 + c] = c < g.dim ? (uint64_t)(uintptr_t)p.v[c] : 0;
    }
    s.arr[6] = (uint64_t)(uintptr_t)p.w;
    return s;
}

template <typename T, int D>
static int sort_keys_perm(const pic_grid_t& g, const pic_particles_t& in, int32_t* perm, int32_t* cell_offsets,
                          const SortWs& ws, bool chained, cudaStream_t st, uint32_t* holes = nullptr, int* sorted_src = nullptr)
{
    // holes != NULL (launch_sort_inplace): the movers' positions, in position order, are copied there before the radix
    // passes; every pass keeps its (key, position) lists (*sorted_src = the buffer that ends up sorted); perm is not written
    const int64_t n = in.n;
    const int C = (int)ws.nkeys;                      // cells, or buckets (pic_sort_buckets)
    mark_phase(PIC_PHASE_BEGIN, st);
    PIC_CUDA_OK(cudaMemsetAsync(ws.zero_begin, 0, ws.zero_bytes, st));
    // the hint: cell_offsets as found on entry -- or, in a chain, what the previous step left in the workspace
    k_hint_hist<<<(unsigned)((C + 1 + 255) / 256), 256, 0, st>>>(cell_offsets, ws.prev_off, ws.chain_sig, chain_sig_of(g, in),
                                                                 chained ? 1 : 0, ws.old_off, C, n, ws.counters, ws.emit.cell_out,
                                                                 ws.emit.mover_in, ws.cell_count, ws.mover_count, ws.mover_lo);
    count_launch();
    if (n > 0) {
        // not a chain: keys, histograms and the stayer/mover split from the positions.  Movers are staged per tile in
        // the second halves of the ping-pong arrays, then packed
        auto classify = ws.bucket ? k_classify<T, D, true> : k_classify<T, D, false>;
        classify<<<(unsigned)ws.cls_tiles, kClsThreads, 0, st>>>(
            make_partp<T>(in), make_gridp<T>(g, ws.bucket), (int)n, ws.old_off, ws.cell_count, ws.mover_count, ws.mover_lo, ws.keys[1],
            ws.idx[1], ws.mask, ws.mprefix, ws.tile_count, ws.pkey, ws.counters);
        k_scan_cells<<<(unsigned)((ws.stage_tiles + kScanTile - 1) / kScanTile), kScanThreads, 0, st>>>(
            ws.tile_count, ws.tile_base, (int)ws.stage_tiles, ws.cls_status, ws.counters + kCtrCls, nullptr, 0, 0);
        k_movers_place<<<(unsigned)ws.stage_tiles, 256, 0, st>>>(ws.keys[1], ws.idx[1], ws.keys[0], ws.idx[0], ws.mask,
                                                                ws.mprefix, ws.tile_base, (int)ws.stage_tiles, n, ws.counters,
                                                                ws.chain_sig);
        count_launch(3);
        if (holes) PIC_CUDA_OK(cudaMemcpyAsync(holes, ws.idx[0], sizeof(uint32_t) * (size_t)n, cudaMemcpyDeviceToDevice, st));
    } else {
        PIC_CUDA_OK(cudaMemsetAsync(ws.hist_begin, 0, ws.hist_bytes, st));
    }
    mark_phase(PIC_PHASE_KEYS, st);
    k_scan_cells<<<(unsigned)ws.scan_tiles, kScanThreads, 0, st>>>(ws.cell_count, cell_offsets, C, ws.scan_status,
                                                                    ws.counters + kCtrScanA, nullptr, 0, 0, ws.prev_off);
    count_launch();
    if (n > 0) {
        k_scan_cells<<<(unsigned)ws.scan_tiles, kScanThreads, 0, st>>>(ws.mover_count, ws.mover_off, C,
                                                                        ws.scan_status + ws.scan_tiles, ws.counters + kCtrScanB,
                                                                        ws.digit_hist, ws.passes, ws.bits_per_pass);
        k_scan_digits<<<ws.passes, kRadix, 0, st>>>(ws.digit_hist);
        const int64_t pass_stride = ws.radix_tiles * kRadix;
        k_zero_lookback<<<sm_count() * 4, 256, 0, st>>>(ws.lookback, ws.counters, ws.passes, pass_stride);
        count_launch(3);
        mark_phase(PIC_PHASE_SCAN, st);
        int src = 0;
        const PermP pp{cell_offsets, ws.mover_off, ws.old_off, perm};
        for (int q = 0; q < ws.passes; ++q) {
            auto kern = (!holes && q == ws.passes - 1) ? k_radix_pass<true> : k_radix_pass<false>;
            kern<<<(unsigned)ws.radix_tiles, kRadixThreads, 0, st>>>(
                ws.keys[src], ws.idx[src], ws.keys[src ^ 1], ws.idx[src ^ 1], ws.counters, q * ws.bits_per_pass,
                (1u << ws.bits_per_pass) - 1u, ws.digit_hist + q * kRadix, ws.counters + kCtrRadix + q,
                ws.lookback + (size_t)q * (size_t)pass_stride, pp);
            count_launch();
            src ^= 1;
        }
        mark_phase(PIC_PHASE_RADIX, st);
        if (sorted_src) *sorted_src = src;
        if (holes) {
            mark_phase(PIC_PHASE_REORDER, st);
            return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
        }
        k_cell_base<<<(unsigned)((C + 255) / 256), 256, 0, st>>>(cell_offsets, ws.old_off, ws.mover_lo, ws.mask, ws.mprefix,
                                                                 ws.cell_base, C, ws.counters);
        k_perm_stayers<<<(unsigned)((n + 256 * kStayIPT - 1) / (256 * kStayIPT)), 256, 0, st>>>(
            ws.pkey, ws.cell_base, ws.mask, ws.mprefix, perm, (int)n, ws.counters);
        count_launch(2);
    }
    mark_phase(PIC_PHASE_REORDER, st);
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

template <typename T, int D>
static int sort_impl(const pic_grid_t& g, const pic_particles_t& in, pic_particles_t& out, int32_t* perm,
                     int32_t* cell_offsets, const SortWs& ws, bool reorder, bool chained, cudaStream_t st)
{
    int rc = sort_keys_perm<T, D>(g, in, perm, cell_offsets, ws, chained, st);
    if (rc != PIC_OK) return rc;
    const int64_t n = in.n;
    if (n > 0 && reorder) {
        // most particles stay where they are: gather value by value; most of them move (first sort): 32-byte records
        if ((rc = launch_reorder(g, in, out, perm, ws.gate, 0u, st)) != PIC_OK) return rc;
        return launch_reorder_records(g, in, out, perm, ws.rec_scratch, ws.gate, 1u, st);
    }
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

// ----------------------------------------------------------------------------- Alg. 2: in place, only misplaced particles move
// "Bucketsort for pre-ordered particles, contiguous datastructure" (Alg. 2; 190-196; the sort the
// paper prefers).  bucket_sizes and bucket_offsets first (l.1-5: k_keys_hist, k_scan_cells); a particle
// is MISPLACED if its position lies outside the region [offsets[key], offsets[key+1]) of its own key (l.6-17:
// bucket_num[ip] != key) -- which is this file's stayer/mover split with the NEW offsets as the hint, so k_classify and
// the movers' radix sort do l.13-30: the movers in position order are the holes_buffer (regions are ordered by
// position), the movers sorted stably by key are the particles_buffer (grouped by target bucket); l.31-35: buffer
// entry i goes into hole i (reading R24: slots in ascending position; the paper's atomic counters leave it open).
template <typename T, int D, bool BK>
__global__ void __launch_bounds__(256) k_keys_hist(PartP<T> p, GridP<T> g, int n, int32_t* __restrict__ count)
{
    const int lane = threadIdx.x & 31;
    for (int base = (blockIdx.x * blockDim.x + threadIdx.x) & ~31; base < n; base += gridDim.x * blockDim.x) {
        const int i = base + lane;
        int key = -1;
        if (i < n) {
            int cell[3] = {0, 0, 0};
#pragma unroll
            for (int c = 0; c < D; ++c) cell[c] = cell_index(grid_coord(p.x[c][i], g.h[c], g.inv_h[c], g.hmul), g.n[c]);
            key = sort_key<T, D, BK>(g, cell);
        }
        const unsigned peers = __match_any_sync(0xFFFFFFFFu, key);       // one atomic per distinct key of the warp
        if (key >= 0 && lane == __ffs(peers) - 1) atomicAdd(&count[key], __popc(peers));
    }
}

template <typename T>
__global__ void __launch_bounds__(256) k_alg2_gather(RecPtrs<T> a, T* __restrict__ buf, int64_t stride, const uint32_t* __restrict__ sorted_idx,
                                                     const uint32_t* __restrict__ counters)
{
    const int64_t m = counters[kCtrMovers];
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < m; i += (int64_t)gridDim.x * blockDim.x) {
        const uint32_t from = sorted_idx[i];
#pragma unroll
        for (int k = 0; k < 7; ++k)
            if (a.s[k]) buf[k * stride + i] = a.s[k][from];
    }
}

template <typename T>
__global__ void __launch_bounds__(256) k_alg2_scatter(RecPtrs<T> a, const T* __restrict__ buf, int64_t stride, const uint32_t* __restrict__ holes,
                                                      const uint32_t* __restrict__ counters, int32_t* __restrict__ moved)
{
    const int64_t m = counters[kCtrMovers];
    if (moved && blockIdx.x == 0 && threadIdx.x == 0) *moved = (int32_t)m;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < m; i += (int64_t)gridDim.x * blockDim.x) {
        const uint32_t to = holes[i];
#pragma unroll
        for (int k = 0; k < 7; ++k)
            if (a.d[k]) a.d[k][to] = buf[k * stride + i];
    }
}

template <typename T, int D>
static int sort_inplace_impl(const pic_grid_t& g, const pic_particles_t& p, int32_t* offsets, const SortWs& ws, void* buffer,
                             int32_t* moved, cudaStream_t st)
{
    const int64_t n = p.n;
    const int C = (int)ws.nkeys;
    // l.1-5: histogram and prefix sum -> the offsets, which are then the hint of the split below
    PIC_CUDA_OK(cudaMemsetAsync(ws.zero_begin, 0, ws.zero_bytes, st));
    PIC_CUDA_OK(cudaMemsetAsync(ws.hist_begin, 0, ws.hist_bytes, st));
    if (n > 0) {
        const int64_t want_blocks = (n + 255) / 256, cap = (int64_t)sm_count() * 16;
        auto kh = ws.bucket ? k_keys_hist<T, D, true> : k_keys_hist<T, D, false>;
        kh<<<(unsigned)(want_blocks < cap ? want_blocks : cap), 256, 0, st>>>(make_partp<T>(p), make_gridp<T>(g, ws.bucket), (int)n, ws.cell_count);
        count_launch();
    }
    k_scan_cells<<<(unsigned)ws.scan_tiles, kScanThreads, 0, st>>>(ws.cell_count, offsets, C, ws.scan_status, ws.counters + kCtrScanA,
                                                                    nullptr, 0, 0);
    count_launch();
    // l.6-30: misplaced particles (position outside the region of their key), in position order and sorted by key
    int src = 0;
    int rc = sort_keys_perm<T, D>(g, p, nullptr, offsets, ws, false, st, ws.pkey, &src);
    if (rc != PIC_OK) return rc;
    if (n > 0) {                                       // l.31-35 through the particles_buffer
        RecPtrs<T> rp;
        int A = 0;
        for (int k = 0; k < 8; ++k) { rp.s[k] = nullptr; rp.d[k] = nullptr; }
        for (int c = 0; c < g.dim; ++c) { rp.s[A] = (const T*)p.x[c]; rp.d[A++] = (T*)p.x[c]; }
        for (int c = 0; c < g.dim; ++c) { rp.s[A] = (const T*)p.v[c]; rp.d[A++] = (T*)p.v[c]; }
        rp.s[A] = (const T*)p.w; rp.d[A++] = (T*)p.w;
        const unsigned blocks = (unsigned)(sm_count() * 8);
        k_alg2_gather<T><<<blocks, 256, 0, st>>>(rp, (T*)buffer, n, ws.idx[src], ws.counters);
        k_alg2_scatter<T><<<blocks, 256, 0, st>>>(rp, (const T*)buffer, n, ws.pkey, ws.counters, moved);
        count_launch(2);
    } else if (moved) {
        PIC_CUDA_OK(cudaMemsetAsync(moved, 0, sizeof(int32_t), st));
    }
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

int launch_sort_inplace(const pic_grid_t& g, const pic_particles_t& p, int32_t* offsets, const SortWs& ws, void* buffer,
                        int32_t* moved, cudaStream_t st)
{
    if (g.dtype == PIC_F32)
        return g.dim == 2 ? sort_inplace_impl<float, 2>(g, p, offsets, ws, buffer, moved, st)
                          : sort_inplace_impl<float, 3>(g, p, offsets, ws, buffer, moved, st);
    return g.dim == 2 ? sort_inplace_impl<double, 2>(g, p, offsets, ws, buffer, moved, st)
                      : sort_inplace_impl<double, 3>(g, p, offsets, ws, buffer, moved, st);
}

// the next call may chain on to the step that has just been enqueued on `out`
int launch_chain_commit(const pic_grid_t& g, const pic_particles_t& out, const SortWs& ws, cudaStream_t st)
{
    k_chain_commit<<<1, 1, 0, st>>>(ws.chain_sig, chain_sig_of(g, out));
    count_launch();
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

int launch_reorder(const pic_grid_t& g, const pic_particles_t& in, const pic_particles_t& out, const int32_t* perm,
                   const uint32_t* gate, uint32_t want, cudaStream_t st)
{
    const int64_t n = in.n;
    if (n <= 0) return PIC_OK;
    // a grid-stride loop over a fixed grid (8 blocks per multiprocessor): cheap to launch when the gate says no
    const int64_t want_blocks = (n + 255) / 256, cap = (int64_t)sm_count() * 8;
    const unsigned blocks = (unsigned)(want_blocks < cap ? want_blocks : cap);
    if (g.dtype == PIC_F32) {
        if (g.dim == 2) k_reorder<float, 2><<<blocks, 256, 0, st>>>(make_partp<float>(in), make_partp<float>(out), perm, n, gate, want);
        else k_reorder<float, 3><<<blocks, 256, 0, st>>>(make_partp<float>(in), make_partp<float>(out), perm, n, gate, want);
    } else {
        if (g.dim == 2) k_reorder<double, 2><<<blocks, 256, 0, st>>>(make_partp<double>(in), make_partp<double>(out), perm, n, gate, want);
        else k_reorder<double, 3><<<blocks, 256, 0, st>>>(make_partp<double>(in), make_partp<double>(out), perm, n, gate, want);
    }
    count_launch();
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

int launch_sort(const pic_grid_t& g, const pic_particles_t& in, pic_particles_t& out, int32_t* perm,
                int32_t* cell_offsets, const SortWs& ws, bool reorder, bool chained, cudaStream_t st)
{
    if (g.dtype == PIC_F32) {
        return g.dim == 2 ? sort_impl<float, 2>(g, in, out, perm, cell_offsets, ws, reorder, chained, st)
                          : sort_impl<float, 3>(g, in, out, perm, cell_offsets, ws, reorder, chained, st);
    }
    return g.dim == 2 ? sort_impl<double, 2>(g, in, out, perm, cell_offsets, ws, reorder, chained, st)
                      : sort_impl<double, 3>(g, in, out, perm, cell_offsets, ws, reorder, chained, st);
}

}  // namespace pic
