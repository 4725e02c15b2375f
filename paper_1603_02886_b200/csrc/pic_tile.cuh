// pic_tile.cuh -- the sorted-order kernel: deposit and/or gather+accel+push over particles that
// are grouped by cell (rows a5-a7, their fusion a8, optionally fused with the reorder a4).
//
// Prior art: the paper's CUDA kernel stages a per-block tile of rho in shared memory and
// atomicAdds every particle's 8 products into it ("sorting is required"),
// and notes the alternative of reducing "on a temporary thread-private variable without atomics",
// putting the result "only once with atomic adds to the grid".  On sm_100a a
// floating-point atomicAdd on shared memory is a compare-and-swap loop (ATOMS.CAST.SPIN, about 5
// lanes per clock per SM against 128 for FFMA), so this kernel takes the second road,
// and what it stages in shared memory is the PARTICLES, not the grid:
//
//   1. a block owns kTile consecutive slots of the sorted order.  All threads copy the block's
//      particles into shared memory (through perm when the reorder is fused in: slot j holds
//      particle perm[j] of src), several independent loads in flight per thread.
//   2. the block lists the cell runs inside its tile ("items", at most kItemMax particles each).
//   3. a GROUP of G lanes owns one item.  Every lane keeps the S^d node sums of its own particles
//      in registers (thread-private); the field stencil of the cell (S^d nodes x d components) is
//      staged once per item in the group's shared-memory slot and read back by broadcast 128-bit
//      loads, NB particles per lane at a time.  New x, v overwrite the particle in shared memory.
//   4. at the end of the item the G lanes combine their sums with a transposed butterfly of
//      shuffles (lane l ends up with the totals of nodes l, l+G, ...: consecutive lanes hold
//      consecutive nodes of a grid row) and add them to the grid with global reductions (RED), in
//      double precision, so that the result does not depend on the density (config 4).
//   5. the block writes its tile back with coalesced 128-bit stores.
//
// S = stencil width of a CELL: 2 for p = 1, 4 for p = 2, 3 (a quadratic particle touches 3 of the
// 4 nodes i0-1..i0+2, which 3 depends on xi >= 1/2; the fourth weight is an exact zero).
// Arithmetic on pairs of x-neighbouring nodes uses the packed fp32 instructions of sm_100
// (fma.rn.f32x2): same FMA-pipe time, half the issue slots.
#pragma once
#include "pic_common.cuh"

namespace pic {

template <typename T>
struct FieldP {
    const T* E[3];
};

enum { kModeDeposit = 1, kModePush = 2, kModeBoth = 3 };

#ifndef PIC_TILE_THREADS
#define PIC_TILE_THREADS 128
#endif
constexpr int kTileThreads = PIC_TILE_THREADS;
constexpr int kG = 8;                  // lanes per item

template <typename T>
struct TileShape {
    static constexpr int kTile = (sizeof(T) == 4 ? 1792 : 1024) * kTileThreads / 128;   // particles per block (3 resident blocks of fp32)
    static constexpr int NB = sizeof(T) == 4 ? 2 : 1;            // particles per lane and batch
};

template <int P>
struct StencilW {
    static constexpr int S = (P == 1) ? 2 : 4;
};

// ---------------------------------------------------------------------------------------------
// packed pairs: fp32 pairs live in one 64-bit register and use the f32x2 instructions
template <typename T>
struct Pk;
template <>
struct Pk<float> {
    unsigned long long r;
};
template <>
struct Pk<double> {
    double lo, hi;
};

__device__ __forceinline__ Pk<float> pk_make(float lo, float hi)
{
    Pk<float> p;
    asm("mov.b64 %0, {%1, %2};" : "=l"(p.r) : "f"(lo), "f"(hi));
    return p;
}
__device__ __forceinline__ Pk<double> pk_make(double lo, double hi) { return Pk<double>{lo, hi}; }
__device__ __forceinline__ float pk_lo(Pk<float> p)
{
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p.r));
    return lo;
}
__device__ __forceinline__ float pk_hi(Pk<float> p)
{
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p.r));
    return hi;
}
__device__ __forceinline__ double pk_lo(Pk<double> p) { return p.lo; }
__device__ __forceinline__ double pk_hi(Pk<double> p) { return p.hi; }
__device__ __forceinline__ Pk<float> pk_fma(Pk<float> a, Pk<float> b, Pk<float> c)
{
    Pk<float> d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d.r) : "l"(a.r), "l"(b.r), "l"(c.r));
    return d;
}
__device__ __forceinline__ Pk<double> pk_fma(Pk<double> a, Pk<double> b, Pk<double> c)
{
    return Pk<double>{fma(a.lo, b.lo, c.lo), fma(a.hi, b.hi, c.hi)};
}
__device__ __forceinline__ Pk<float> pk_mul(Pk<float> a, Pk<float> b)
{
    Pk<float> d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d.r) : "l"(a.r), "l"(b.r));
    return d;
}
__device__ __forceinline__ Pk<double> pk_mul(Pk<double> a, Pk<double> b) { return Pk<double>{a.lo * b.lo, a.hi * b.hi}; }
template <typename T>
__device__ __forceinline__ Pk<T> pk_zero()
{
    return pk_make((T)0, (T)0);
}

// weights of one particle on the S-wide stencil of its cell; returns the (clamped) cell index
template <typename T, int P>
__device__ __forceinline__ int cell_weights(T x, T h, T inv_h, int hmul, int n, T (&w)[StencilW<P>::S])
{
    const T t = grid_coord(x, h, inv_h, hmul);
    const int i0 = cell_index(t, n);
    const T xi = t - (T)i0;
    if constexpr (P == 1) {
        w[0] = (T)1 - xi;
        w[1] = xi;
    } else if constexpr (P == 2) {
        const bool up = xi >= (T)0.5;
        const T d = xi - (up ? (T)1 : (T)0);
        const T a = (T)0.5 - d, b = (T)0.5 + d;
        const T w0 = (T)0.5 * a * a, w1 = (T)0.75 - d * d, w2 = (T)0.5 * b * b;
        w[0] = up ? (T)0 : w0;
        w[1] = up ? w0 : w1;
        w[2] = up ? w1 : w2;
        w[3] = up ? w2 : (T)0;
    } else {
        const T om = (T)1 - xi, x2 = xi * xi;
        w[0] = om * om * om * (T)(1.0 / 6.0);
        w[1] = (T)(2.0 / 3.0) - x2 + (T)0.5 * x2 * xi;
        w[2] = (T)(1.0 / 6.0) + (T)0.5 * (xi + x2 - x2 * xi);
        w[3] = x2 * xi * (T)(1.0 / 6.0);
    }
    return i0;
}

// S consecutive values from shared memory as S/2 pairs (128-bit loads)
template <typename T, int S>
__device__ __forceinline__ void load_row(const T* __restrict__ p, Pk<T> (&e)[S / 2])
{
    if constexpr (sizeof(T) == 4 && S == 4) {
        const float4 v = *reinterpret_cast<const float4*>(p);
        e[0] = pk_make(v.x, v.y);
        e[1] = pk_make(v.z, v.w);
    } else if constexpr (sizeof(T) == 4) {
        const float2 v = *reinterpret_cast<const float2*>(p);
        e[0] = pk_make(v.x, v.y);
    } else {
#pragma unroll
        for (int i = 0; i < S / 2; ++i) {
            const double2 v = *reinterpret_cast<const double2*>(p + 2 * i);
            e[i] = pk_make(v.x, v.y);
        }
    }
}

// Combine the per-lane node sums of a group of G lanes (transposed butterfly).  NODES and G are
// powers of two.  With GS = min(G, NODES): afterwards acc[a], a < NODES/GS, holds the group total
// of node a*GS + (lg % GS); `owner` is false on lanes whose totals duplicate another lane's
// (only when NODES < G).
template <typename T, int NODES, int G>
__device__ __forceinline__ void group_combine(T (&acc)[NODES], int lg, bool& owner)
{
    owner = true;
    int cnt = NODES;
#pragma unroll
    for (int m = 1; m < G; m <<= 1) {
        const bool upper = (lg & m) != 0;
        if (cnt >= 2) {
            const int half = cnt / 2;
#pragma unroll
            for (int a = 0; a < NODES / 2; ++a) {
                if (a < half) {
                    const T send = upper ? acc[2 * a] : acc[2 * a + 1];
                    const T keep = upper ? acc[2 * a + 1] : acc[2 * a];
                    acc[a] = keep + __shfl_xor_sync(0xFFFFFFFFu, send, m);
                }
            }
            cnt = half;
        } else {
            acc[0] += __shfl_xor_sync(0xFFFFFFFFu, acc[0], m);
            owner = owner && !upper;
        }
    }
}

// One particle of the tile whose cell is not the cell of the run it sits in (cell_offsets that do
// not describe the order): the paper's threads-on-particles path (3.3.4) with direct
// global reductions and read-only loads.  Reads and writes slot `slot` of the staged tile.
template <typename T, int D, int P, int MODE>
__device__ __forceinline__ void stray_particle(T* __restrict__ sp, int tile_stride, int slot, const GridP<T>& g,
                                               const FieldP<T>& f, double* __restrict__ racc, T dt, T qmdt)
{
    int first[3] = {0, 0, 0};
    T wt[3][P + 1];
    T x[D];
#pragma unroll
    for (int c = 0; c < D; ++c) {
        x[c] = sp[c * tile_stride + slot];
        T t = grid_coord(x[c], g.h[c], g.inv_h[c], g.hmul);
        spline_weights<T, P>(t, cell_index(t, g.n[c]), first[c], wt[c]);
    }
    T e[D];
#pragma unroll
    for (int c = 0; c < D; ++c) e[c] = (T)0;
    T q = (T)0;
    if (MODE & kModeDeposit) q = sp[2 * D * tile_stride + slot] * g.inv_vol;
    constexpr int PZ = (D == 3) ? P : 0;
#pragma unroll
    for (int cz = 0; cz <= PZ; ++cz) {
        const int jz = (D == 3) ? fold(first[2] + cz, g.n[2]) : 0;
        const T wz = (D == 3) ? wt[2][cz] : (T)1;
#pragma unroll
        for (int b = 0; b <= P; ++b) {
            const int jy = fold(first[1] + b, g.n[1]);
            const T wyz = wz * wt[1][b];
            const int64_t row = (int64_t)g.n[0] * (jy + (int64_t)g.n[1] * jz);
#pragma unroll
            for (int a = 0; a <= P; ++a) {
                const int jx = fold(first[0] + a, g.n[0]);
                const T wgt = wyz * wt[0][a];
                if (MODE & kModeDeposit) atomicAdd(&racc[row + jx], (double)(q * wgt));
                if (MODE & kModePush) {
#pragma unroll
                    for (int c = 0; c < D; ++c) e[c] += wgt * __ldg(f.E[c] + row + jx);
                }
            }
        }
    }
    if (MODE & kModePush) {
#pragma unroll
        for (int c = 0; c < D; ++c) {
            const T v = sp[(D + c) * tile_stride + slot] + qmdt * e[c];
            sp[(D + c) * tile_stride + slot] = v;
            sp[c * tile_stride + slot] = wrap_periodic(x[c] + dt * v, g.L[c], g.inv_L[c]);
        }
    }
}

template <typename T, int D, int P>
struct TileSmem {
    static constexpr int S = StencilW<P>::S;
    static constexpr int NODES = (D == 3) ? S * S * S : S * S;
    static constexpr int A = 2 * D + 1;
    static constexpr int kTile = TileShape<T>::kTile;
    static constexpr int GROUPS = kTileThreads / kG;
    static constexpr int EPAD = 16 / sizeof(T);                   // shifts consecutive groups by four banks
    static constexpr int ESTRIDE = D * NODES + EPAD;
    static constexpr int kItemMax = 16 * kG * TileShape<T>::NB;
    static constexpr int kMaxItems = kTile + kTile / kItemMax + 2;
    static constexpr size_t part_bytes = sizeof(T) * A * kTile;
    static constexpr size_t field_bytes = sizeof(T) * GROUPS * ESTRIDE;
    static constexpr size_t item_bytes = sizeof(uint32_t) * kMaxItems;               // (start, len) per item
    static constexpr size_t order_bytes = (sizeof(uint16_t) * kMaxItems + 15) / 16 * 16;  // items, longest first
    static constexpr size_t stray_bytes = sizeof(uint32_t) * (kTile / 32);          // one bit per slot
    static constexpr size_t bytes(int mode)
    {
        return part_bytes + ((mode & kModePush) ? field_bytes : 0) + item_bytes + order_bytes + stray_bytes;
    }
};

template <typename T, int D, int P, int MODE>
constexpr int tile_min_blocks()
{
    // resident blocks per SM the kernel is compiled for (register budget 65536 / (128 * blocks))
    return ((sizeof(T) == 4) ? 3 : 1) * (128 / kTileThreads);
}

template <typename T, int D, int P, int MODE, bool VIA_PERM>
__global__ void __launch_bounds__(kTileThreads, (tile_min_blocks<T, D, P, MODE>()))
k_tile(PartP<T> src, PartP<T> dst, const int32_t* __restrict__ perm, GridP<T> g, FieldP<T> f,
       const int32_t* __restrict__ cell_offsets, int64_t n, double* __restrict__ racc, T dt, T qmdt)
{
    using SM = TileSmem<T, D, P>;
    constexpr int S = SM::S, S2 = S / 2;
    constexpr int SZ = (D == 3) ? S : 1;
    constexpr int NODES = SM::NODES;
    constexpr int A = SM::A;
    constexpr int kTile = SM::kTile;
    constexpr int G = kG;
    constexpr int NB = TileShape<T>::NB;
    constexpr int GPW = 32 / G;                        // groups per warp
    constexpr int kItemMax = SM::kItemMax;
    constexpr int GS = (G < NODES) ? G : NODES;        // lanes of a group that own distinct nodes
    constexpr int NPL = NODES / GS;                    // nodes per lane after the combine
    constexpr bool DEP = (MODE & kModeDeposit) != 0, PUSH = (MODE & kModePush) != 0;
    constexpr unsigned FULL = 0xFFFFFFFFu;
    constexpr int VEC = 16 / sizeof(T);                // elements per 128-bit access

    extern __shared__ __align__(16) unsigned char s_dyn[];
    T* const sp = reinterpret_cast<T*>(s_dyn);                                        // [A][kTile]
    T* const sE = reinterpret_cast<T*>(s_dyn + SM::part_bytes);                       // [GROUPS][ESTRIDE]
    uint32_t* const s_item = reinterpret_cast<uint32_t*>(s_dyn + SM::part_bytes + (PUSH ? SM::field_bytes : 0));
    uint16_t* const s_order = reinterpret_cast<uint16_t*>(reinterpret_cast<unsigned char*>(s_item) + SM::item_bytes);
    uint32_t* const s_stray = reinterpret_cast<uint32_t*>(reinterpret_cast<unsigned char*>(s_order) + SM::order_bytes);
    constexpr int kClasses = 16;                // items are queued by number of batches, longest first
    __shared__ int s_cls[kClasses + 1];
    __shared__ int s_cells[2];
    __shared__ int s_nitems, s_next, s_anystray;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lg = lane % G;                    // lane within the group
    const int gid = tid / G;                    // group within the block
    const int64_t j0 = (int64_t)blockIdx.x * kTile;
    const int cnt = (int)((n - j0 < (int64_t)kTile) ? (n - j0) : (int64_t)kTile);

    // ---- 1. stage the tile: slot j <- particle (perm[j0+j] | j0+j), VEC slots per thread and round.
    //         Row a of the staged tile: x[a] for a < D, v[a-D] for a < 2D, w for a == 2D.
    auto needed = [](int a) { return a < D || (a < 2 * D ? (PUSH || VIA_PERM) : (DEP || VIA_PERM)); };
    auto src_row = [&](int a) -> const T* { return a < D ? src.x[a] : (a < 2 * D ? src.v[a - D] : src.w); };
    if constexpr (VIA_PERM) {
        // consecutive lanes take consecutive slots: particles that kept their cell sit in runs of
        // consecutive source indices, so most of a warp's 32 loads fall into one or two lines
        constexpr int U = 4;                    // slots per thread in flight (U perm words, then U*A loads)
        for (int q0 = 0; q0 < cnt; q0 += kTileThreads * U) {
            int idx[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int q = q0 + u * kTileThreads + tid;
                idx[u] = q < cnt ? perm[j0 + q] : -1;
            }
            T val[A][U];
#pragma unroll
            for (int a = 0; a < A; ++a) {
                if (!needed(a)) continue;
                const T* arr = src_row(a);
#pragma unroll
                for (int u = 0; u < U; ++u)
                    if (idx[u] >= 0) val[a][u] = arr[idx[u]];
            }
#pragma unroll
            for (int a = 0; a < A; ++a) {
                if (!needed(a)) continue;
#pragma unroll
                for (int u = 0; u < U; ++u)
                    if (idx[u] >= 0) sp[a * kTile + q0 + u * kTileThreads + tid] = val[a][u];
            }
        }
    } else {
        for (int q = tid * VEC; q < cnt; q += kTileThreads * VEC) {
            if (q + VEC <= cnt) {
                T val[A][VEC];
#pragma unroll
                for (int a = 0; a < A; ++a) {
                    if (!needed(a)) continue;
                    const T* arr = src_row(a);
                    if constexpr (VEC == 4) {
                        const float4 v4 = *reinterpret_cast<const float4*>(arr + j0 + q);
                        val[a][0] = v4.x; val[a][1] = v4.y; val[a][2] = v4.z; val[a][3] = v4.w;
                    } else {
                        const double2 v2 = *reinterpret_cast<const double2*>(arr + j0 + q);
                        val[a][0] = v2.x; val[a][1] = v2.y;
                    }
                }
#pragma unroll
                for (int a = 0; a < A; ++a) {
                    if (!needed(a)) continue;
                    if constexpr (VEC == 4)
                        *reinterpret_cast<float4*>(sp + a * kTile + q) = make_float4(val[a][0], val[a][1], val[a][2], val[a][3]);
                    else
                        *reinterpret_cast<double2*>(sp + a * kTile + q) = make_double2(val[a][0], val[a][1]);
                }
            } else {
                for (int e = 0; q + e < cnt; ++e) {
#pragma unroll
                    for (int a = 0; a < A; ++a)
                        if (needed(a)) sp[a * kTile + q + e] = src_row(a)[j0 + q + e];
                }
            }
        }
    }
    for (int i = tid; i < kTile / 32; i += kTileThreads) s_stray[i] = 0u;
    if (tid <= kClasses) s_cls[tid] = 0;
    if (tid == 0) { s_nitems = 0; s_next = 0; s_anystray = 0; }
    __syncthreads();

    // ---- 2. cells whose runs (by cell_offsets) hold the first and the last slot of the tile: the key
    //         of that particle if the order is consistent, else a binary search; then the item list:
    //         every cell's run inside the tile, cut into pieces of at most kItemMax
    if (tid < 2) {
        const int slot = tid == 0 ? 0 : cnt - 1;
        const int64_t j = j0 + slot;
        int k = 0, mul = 1;
#pragma unroll
        for (int c = 0; c < D; ++c) {
            T t = grid_coord(sp[c * kTile + slot], g.h[c], g.inv_h[c], g.hmul);
            k += mul * cell_index(t, g.n[c]);
            mul *= g.n[c];
        }
        if (!((int64_t)cell_offsets[k] <= j && j < (int64_t)cell_offsets[k + 1])) {
            int lo = 0, hi = mul;                       // largest k with cell_offsets[k] <= j
            while (hi - lo > 1) {
                const int mid = lo + (hi - lo) / 2;
                if ((int64_t)cell_offsets[mid] <= j) lo = mid; else hi = mid;
            }
            k = lo;
        }
        s_cells[tid] = k;
    }
    __syncthreads();
    {
        const int c_first = s_cells[0], c_last = s_cells[1];
        const int64_t j1 = j0 + cnt;
        for (int c = c_first + tid; c <= c_last; c += kTileThreads) {
            const int64_t a = cell_offsets[c], b = cell_offsets[c + 1];
            const int64_t lo = a > j0 ? a : j0, hi = b < j1 ? b : j1;
            const int s = (int)(lo - j0);
            const int len = hi > lo ? (int)(hi - lo) : 0;
            const int nch = (len + kItemMax - 1) / kItemMax;
            if (nch > 0) {
                const int pos = atomicAdd(&s_nitems, nch);
                for (int q = 0; q < nch; ++q) {
                    if (pos + q < SM::kMaxItems) {
                        const int rem = len - q * kItemMax;
                        const int l = rem < kItemMax ? rem : kItemMax;
                        s_item[pos + q] = (uint32_t)(s + q * kItemMax) | ((uint32_t)l << 16);
                        atomicAdd(&s_cls[kClasses - (l + G * NB - 1) / (G * NB)], 1);   // class 0 = longest
                    }
                }
            }
        }
        __syncthreads();
        if (tid == 0) {                         // exclusive prefix over the classes
            int run = 0;
            for (int k = 0; k <= kClasses; ++k) { const int c = s_cls[k]; s_cls[k] = run; run += c; }
            if (s_nitems > SM::kMaxItems) s_nitems = SM::kMaxItems;
        }
        __syncthreads();
        for (int i = tid; i < s_nitems; i += kTileThreads) {
            const int l = (int)(s_item[i] >> 16);
            s_order[atomicAdd(&s_cls[kClasses - (l + G * NB - 1) / (G * NB)], 1)] = (uint16_t)i;
        }
        __syncthreads();
    }
    const int nitems = s_nitems;
    T* const myE = sE + gid * SM::ESTRIDE;

    // ---- 3. every warp takes GPW items at a time from the block's queue
    for (;;) {
        int ibase = 0;
        if (lane == 0) ibase = atomicAdd(&s_next, GPW);
        ibase = __shfl_sync(FULL, ibase, 0);
        if (ibase >= nitems) break;
        const int item = ibase + lane / G;
        const bool have = item < nitems;
        const uint32_t it = have ? s_item[s_order[item]] : 0u;
        const int start = (int)(it & 0xFFFFu), len = (int)(it >> 16);

        // the item's cell, from its first particle
        int cell[3] = {0, 0, 0};
#pragma unroll
        for (int c = 0; c < D; ++c) {
            T t = grid_coord(sp[c * kTile + start], g.h[c], g.inv_h[c], g.hmul);
            cell[c] = cell_index(t, g.n[c]);
        }
        // grid index of node t*GS + lg%GS of the cell's stencil (the nodes this lane stages and flushes)
        auto node_offset = [&](int t) {
            const int node = t * GS + (lg % GS);
            const int ii = node % S, jj = (node / S) % S, kk = node / (S * S);
            constexpr int sh = (S == 4) ? 1 : 0;
            const int gx = fold(cell[0] - sh + ii, g.n[0]), gy = fold(cell[1] - sh + jj, g.n[1]);
            const int gz = (D == 3) ? fold(cell[2] - sh + kk, g.n[2]) : 0;
            return gx + g.n[0] * (gy + g.n[1] * gz);
        };

        // stage the field stencil of the cell in the group's shared-memory slot
        if constexpr (PUSH) {
            __syncwarp();
            if (have) {
#pragma unroll
                for (int t = 0; t < NPL; ++t) {
                    const int off = node_offset(t);
#pragma unroll
                    for (int c = 0; c < D; ++c) myE[c * NODES + t * GS + (lg % GS)] = __ldg(f.E[c] + off);
                }
            }
            __syncwarp();
        }

        Pk<T> acc[DEP ? NODES / 2 : 1];
#pragma unroll
        for (int a = 0; a < (DEP ? NODES / 2 : 1); ++a) acc[a] = pk_zero<T>();

        // number of batches: warp-uniform
        int nb = (len + G * NB - 1) / (G * NB);
#pragma unroll
        for (int o = 16; o >= G; o >>= 1) nb = max(nb, __shfl_xor_sync(FULL, nb, o));

        for (int bt = 0; bt < nb; ++bt) {
            Pk<T> wx[NB][S2];
            T wy[NB][S], wz[NB][SZ], q[NB];
            int slot[NB];
            bool live[NB];
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int k = (bt * NB + b) * G + lg;
                const bool in_item = k < len;
                slot[b] = start + (in_item ? k : 0);
                T w1[S];
                bool same = cell_weights<T, P>(sp[slot[b]], g.h[0], g.inv_h[0], g.hmul, g.n[0], w1) == cell[0];
#pragma unroll
                for (int i = 0; i < S2; ++i) wx[b][i] = pk_make(w1[2 * i], w1[2 * i + 1]);
                same = (cell_weights<T, P>(sp[kTile + slot[b]], g.h[1], g.inv_h[1], g.hmul, g.n[1], wy[b]) == cell[1]) && same;
                if constexpr (D == 3) {
                    same = (cell_weights<T, P>(sp[2 * kTile + slot[b]], g.h[2], g.inv_h[2], g.hmul, g.n[2], wz[b]) == cell[2]) && same;
                } else {
                    wz[b][0] = (T)1;
                }
                if (in_item && !same) { atomicOr(&s_stray[slot[b] >> 5], 1u << (slot[b] & 31)); s_anystray = 1; }
                live[b] = in_item && same;
                q[b] = (T)0;
                if constexpr (DEP) {
                    if (live[b]) q[b] = sp[2 * D * kTile + slot[b]] * g.inv_vol;
                }
            }

            Pk<T> sg[PUSH ? NB : 1][D][S2];          // gather sums per x-node pair
            if constexpr (PUSH) {
#pragma unroll
                for (int b = 0; b < NB; ++b)
#pragma unroll
                    for (int c = 0; c < D; ++c)
#pragma unroll
                        for (int i = 0; i < S2; ++i) sg[b][c][i] = pk_zero<T>();
            }

#pragma unroll
            for (int kk = 0; kk < SZ; ++kk) {
#pragma unroll
                for (int jj = 0; jj < S; ++jj) {
                    const int row = (kk * S + jj) * S;
                    Pk<T> er[PUSH ? D : 1][S2];
                    if constexpr (PUSH) {
#pragma unroll
                        for (int c = 0; c < D; ++c) load_row<T, S>(myE + c * NODES + row, er[c]);
                    }
#pragma unroll
                    for (int b = 0; b < NB; ++b) {
                        const T wyz = wz[b][kk] * wy[b][jj];
                        if constexpr (DEP) {
                            const T qw = q[b] * wyz;
                            const Pk<T> qw2 = pk_make(qw, qw);
#pragma unroll
                            for (int i = 0; i < S2; ++i) acc[row / 2 + i] = pk_fma(qw2, wx[b][i], acc[row / 2 + i]);
                        }
                        if constexpr (PUSH) {
                            const Pk<T> wyz2 = pk_make(wyz, wyz);
#pragma unroll
                            for (int c = 0; c < D; ++c)
#pragma unroll
                                for (int i = 0; i < S2; ++i) sg[b][c][i] = pk_fma(wyz2, er[c][i], sg[b][c][i]);
                        }
                    }
                }
            }

            if constexpr (PUSH) {
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    if (live[b]) {
#pragma unroll
                        for (int c = 0; c < D; ++c) {
                            Pk<T> t2 = pk_mul(sg[b][c][0], wx[b][0]);
#pragma unroll
                            for (int i = 1; i < S2; ++i) t2 = pk_fma(sg[b][c][i], wx[b][i], t2);
                            const T ec = pk_lo(t2) + pk_hi(t2);
                            const T v = sp[(D + c) * kTile + slot[b]] + qmdt * ec;
                            const T xo = sp[c * kTile + slot[b]];
                            sp[(D + c) * kTile + slot[b]] = v;
                            sp[c * kTile + slot[b]] = wrap_periodic(xo + dt * v, g.L[c], g.inv_L[c]);
                        }
                    }
                }
            }
        }

        // ---- end of the item: combine the G lanes' sums, add the totals to the grid
        if constexpr (DEP) {
            T accs[NODES];
#pragma unroll
            for (int a = 0; a < NODES / 2; ++a) { accs[2 * a] = pk_lo(acc[a]); accs[2 * a + 1] = pk_hi(acc[a]); }
            bool owner;
            group_combine<T, NODES, G>(accs, lg, owner);
            if (have && owner) {
#pragma unroll
                for (int t = 0; t < NPL; ++t) atomicAdd(&racc[node_offset(t)], (double)accs[t]);
            }
        }
    }
    __syncthreads();

    // ---- 4. particles whose cell is not their run's cell (only with inconsistent cell_offsets)
    if (s_anystray) {
        for (int i = tid; i < cnt; i += kTileThreads)
            if ((s_stray[i >> 5] >> (i & 31)) & 1u) stray_particle<T, D, P, MODE>(sp, kTile, i, g, f, racc, dt, qmdt);
        __syncthreads();
    }

    // ---- 5. write the tile back (x, v; w too when the reorder is fused in)
    if constexpr (PUSH || VIA_PERM) {
        constexpr int AS = VIA_PERM ? A : 2 * D;
        const bool full = (cnt == kTile);
#pragma unroll
        for (int a = 0; a < AS; ++a) {
            T* arr = a < D ? dst.x[a] : (a < 2 * D ? dst.v[a - D] : dst.w);
            const T* s = sp + a * kTile;
            if (full) {
                for (int q = tid * VEC; q < kTile; q += kTileThreads * VEC) {
                    if constexpr (VEC == 4)
                        *reinterpret_cast<float4*>(arr + j0 + q) = *reinterpret_cast<const float4*>(s + q);
                    else
                        *reinterpret_cast<double2*>(arr + j0 + q) = *reinterpret_cast<const double2*>(s + q);
                }
            } else {
                for (int q = tid; q < cnt; q += kTileThreads) arr[j0 + q] = s[q];
            }
        }
    }
}

// launch k_tile over n particles sorted by cell.  VIA_PERM: particle perm[j] of src -> slot j of dst;
// otherwise in place on dst (src is ignored).  racc = double accumulation grid of the deposit.
template <typename T, int D, int P, int MODE, bool VIA_PERM>
inline int launch_tile(const pic_grid_t& g, const pic_particles_t& src, const pic_particles_t& dst,
                       const int32_t* perm, const int32_t* cell_offsets, const void* const E[3], double* racc,
                       double dt, double qm, cudaStream_t st)
{
    if (dst.n <= 0) return PIC_OK;
    FieldP<T> f;
    for (int c = 0; c < 3; ++c) f.E[c] = (E && c < D) ? (const T*)E[c] : nullptr;
    auto kern = k_tile<T, D, P, MODE, VIA_PERM>;
    constexpr size_t smem = TileSmem<T, D, P>::bytes(MODE);
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return PIC_ERR_CUDA;
        attr_set = true;
    }
    constexpr int kTile = TileShape<T>::kTile;
    const unsigned blocks = (unsigned)((dst.n + kTile - 1) / kTile);
    kern<<<blocks, kTileThreads, smem, st>>>(make_partp<T>(VIA_PERM ? src : dst), make_partp<T>(dst), perm,
                                            make_gridp<T>(g), f, cell_offsets, dst.n, racc, (T)dt, (T)(qm * dt));
    count_launch();
    return cudaGetLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

// rho[k] = (T) racc[k]
template <typename T>
__global__ void __launch_bounds__(256) k_round_rho(const double* __restrict__ racc, T* __restrict__ rho, int64_t C)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < C) rho[k] = (T)racc[k];
}

}  // namespace pic
