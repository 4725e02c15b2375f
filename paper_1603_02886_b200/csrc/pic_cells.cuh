// pic_cells.cuh -- the sorted-order kernel: deposit and/or gather+accel+push over particles that
// are grouped by cell (rows a5-a7, and their fusion a8, optionally fused with the reorder a4).
//
// Prior art: the paper's CUDA kernel stages a per-block tile of rho in shared memory and
// atomicAdds every particle's 8 products into it ("sorting is required"),
// and notes the alternative of reducing "on a temporary thread-private variable without atomics",
// putting the result "only once with atomic adds to the grid".  On sm_100a a
// floating-point atomicAdd on shared memory is a compare-and-swap loop (ATOMS.CAST.SPIN; measured
// 20x to 600x below FMA throughput), so this kernel takes the second road:
//
//   * a GROUP of G lanes owns one cell's run of particles (an "item", at most kItemMax particles);
//     every lane keeps the S^d node sums of its own particles in registers (thread-private);
//   * at the end of the item the G lanes combine their sums with a transposed butterfly of
//     shuffles (lane l ends up with the totals of nodes l, l+G, l+2G, ...: consecutive lanes hold
//     consecutive nodes of a grid row) and add them to the grid with global reductions (RED) --
//     in double precision, so the result does not depend on the density;
//   * the field stencil of the cell (S^d nodes x d components) is staged once per item in the
//     group's slot of shared memory and read back by broadcast 128-bit loads, NB particles per
//     lane at a time, so one shared-memory word feeds G*NB particles;
//   * warps take items from a block-wide queue, so cells of different population balance out.
//
// S = stencil width of a CELL: 2 for p = 1, 4 for p = 2, 3 (a quadratic particle touches 3 of the
// 4 nodes i0-1..i0+2, which 3 depends on xi >= 1/2; the fourth weight is an exact zero).
//
// With VIA_PERM the kernel reads particle perm[j] of `src` and writes slot j of `dst` (all
// attributes): the reorder of the sort (row a4) happens inside the same pass, the sorted copy at
// time t is never materialised.
#pragma once
#include "pic_common.cuh"

namespace pic {

template <typename T>
struct FieldP {
    const T* E[3];
};

constexpr int kCellThreads = 128;
constexpr int kBlockParticles = 4096;   // sorted particles per block
constexpr int kMaxItems = kBlockParticles;

// resident blocks per SM the kernel is compiled for: the 4^3-node register tile needs ~170 (float)
// or ~250 (double) registers per thread; the smaller stencils fit in 128
template <typename T, int D, int P>
constexpr int cells_min_blocks()
{
    return (D == 3 && P >= 2) ? (sizeof(T) == 4 ? 3 : 2) : 4;
}

enum { kModeDeposit = 1, kModePush = 2, kModeBoth = 3 };

template <int P>
struct StencilW {
    static constexpr int S = (P == 1) ? 2 : 4;
};

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

// row of S consecutive values from shared memory with one (or two) 128-bit loads
template <typename T, int S>
__device__ __forceinline__ void load_row(const T* __restrict__ p, T (&e)[S])
{
    if constexpr (sizeof(T) == 4 && S == 4) {
        const float4 v = *reinterpret_cast<const float4*>(p);
        e[0] = v.x; e[1] = v.y; e[2] = v.z; e[3] = v.w;
    } else if constexpr (sizeof(T) == 4) {
        const float2 v = *reinterpret_cast<const float2*>(p);
        e[0] = v.x; e[1] = v.y;
    } else {
#pragma unroll
        for (int i = 0; i < S; i += 2) {
            const double2 v = *reinterpret_cast<const double2*>(p + i);
            e[i] = v.x; e[i + 1] = v.y;
        }
    }
}

// One particle, any order: direct global reductions and read-only loads (the paper's 3.3.4 path).
// Used for the rare particle of a run whose cell is not the run's cell (inconsistent cell_offsets).
// Reads particle i of src, writes slot j of dst.
template <typename T, int D, int P, int MODE, bool COPY_W>
__device__ __noinline__ void lone_particle(const PartP<T>& src, int64_t i, const PartP<T>& dst, int64_t j,
                                           const GridP<T>& g, const FieldP<T>& f, double* __restrict__ racc, T dt,
                                           T qmdt)
{
    int first[3] = {0, 0, 0};
    T wt[3][P + 1];
    T x[D];
#pragma unroll
    for (int c = 0; c < D; ++c) {
        x[c] = src.x[c][i];
        T t = grid_coord(x[c], g.h[c], g.inv_h[c], g.hmul);
        spline_weights<T, P>(t, cell_index(t, g.n[c]), first[c], wt[c]);
    }
    T e[D];
#pragma unroll
    for (int c = 0; c < D; ++c) e[c] = (T)0;
    T wraw = (T)0;
    if ((MODE & kModeDeposit) || COPY_W) wraw = src.w[i];
    const T q = wraw * g.inv_vol;
    constexpr int PZ = (D == 3) ? P : 0;
    for (int cz = 0; cz <= PZ; ++cz) {
        const int jz = (D == 3) ? fold(first[2] + cz, g.n[2]) : 0;
        const T wz = (D == 3) ? wt[2][cz] : (T)1;
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
            T v = src.v[c][i] + qmdt * e[c];
            dst.v[c][j] = v;
            dst.x[c][j] = wrap_periodic(x[c] + dt * v, g.L[c], g.inv_L[c]);
        }
        if (COPY_W) dst.w[j] = wraw;
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

template <typename T, int D, int P, int MODE, int G, int NB, bool VIA_PERM>
__global__ void __launch_bounds__(kCellThreads, (cells_min_blocks<T, D, P>()))
k_cells(PartP<T> src, PartP<T> dst, const int32_t* __restrict__ perm, GridP<T> g, FieldP<T> f,
        const int32_t* __restrict__ cell_offsets, int64_t n, double* __restrict__ racc, T dt, T qmdt)
{
    constexpr int S = StencilW<P>::S;
    constexpr int SZ = (D == 3) ? S : 1;
    constexpr int NODES = S * S * SZ;
    constexpr int GROUPS = kCellThreads / G;
    constexpr int GPW = 32 / G;                        // groups per warp
    constexpr int kItemMax = 16 * G * NB;              // particles per item
    constexpr int GS = (G < NODES) ? G : NODES;        // lanes of a group that own distinct nodes
    constexpr int NPL = NODES / GS;                    // nodes per lane after the combine
    constexpr bool DEP = (MODE & kModeDeposit) != 0, PUSH = (MODE & kModePush) != 0;
    constexpr unsigned FULL = 0xFFFFFFFFu;
    static_assert(kItemMax <= 65535, "item length is stored in 16 bits");

    extern __shared__ __align__(16) unsigned char s_dyn[];
    T (*s_E)[D][NODES] = reinterpret_cast<T (*)[D][NODES]>(s_dyn);     // [GROUPS][D][NODES] when PUSH
    __shared__ int s_item_start[kMaxItems];
    __shared__ unsigned short s_item_len[kMaxItems];
    __shared__ int s_scan[kCellThreads / 32];
    __shared__ int s_cells[2];
    __shared__ int s_nitems, s_next;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lg = lane % G;                    // lane within the group
    const int gid = tid / G;                    // group within the block
    const int64_t j0 = (int64_t)blockIdx.x * kBlockParticles;
    const int64_t j1 = (j0 + kBlockParticles < n) ? j0 + kBlockParticles : n;

    // ---- cells spanned by this block's particles: keys of the first and the last particle
    if (tid < 2) {
        const int64_t j = tid == 0 ? j0 : j1 - 1;
        const int64_t i = VIA_PERM ? (int64_t)perm[j] : j;
        int k = 0, mul = 1;
#pragma unroll
        for (int c = 0; c < D; ++c) {
            T t = grid_coord(src.x[c][i], g.h[c], g.inv_h[c], g.hmul);
            k += mul * cell_index(t, g.n[c]);
            mul *= g.n[c];
        }
        s_cells[tid] = k;
    }
    if (tid == 0) { s_nitems = 0; s_next = 0; }
    __syncthreads();
    const int c_first = s_cells[0], c_last = s_cells[1];
    // ---- item list: every cell's run inside [j0,j1), cut into pieces of at most kItemMax
    for (int base = c_first; base <= c_last; base += kCellThreads) {
        const int c = base + tid;
        int s = 0, len = 0;
        if (c <= c_last) {
            const int64_t a = cell_offsets[c], b = cell_offsets[c + 1];
            const int64_t lo = a > j0 ? a : j0, hi = b < j1 ? b : j1;
            s = (int)(lo - j0);
            len = hi > lo ? (int)(hi - lo) : 0;
        }
        const int nch = (len + kItemMax - 1) / kItemMax;
        int inc = nch;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(FULL, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) s_scan[warp] = inc;
        __syncthreads();
        int off = s_nitems;
        for (int w = 0; w < warp; ++w) off += s_scan[w];
        const int pos = off + inc - nch;
        for (int q = 0; q < nch; ++q) {
            if (pos + q < kMaxItems) {
                s_item_start[pos + q] = s + q * kItemMax;
                const int rem = len - q * kItemMax;
                s_item_len[pos + q] = (unsigned short)(rem < kItemMax ? rem : kItemMax);
            }
        }
        __syncthreads();
        if (tid == kCellThreads - 1) s_nitems = (off + inc < kMaxItems) ? off + inc : kMaxItems;
        __syncthreads();
    }
    const int nitems = s_nitems;

    // ---- every warp takes GPW items at a time from the block's queue
    for (;;) {
        int ibase = 0;
        if (lane == 0) ibase = atomicAdd(&s_next, GPW);
        ibase = __shfl_sync(FULL, ibase, 0);
        if (ibase >= nitems) break;
        const int item = ibase + lane / G;
        const bool have = item < nitems;
        const int start = have ? s_item_start[item] : 0;
        const int len = have ? (int)s_item_len[item] : 0;
        const int64_t jbeg = j0 + start;

        // the item's cell, from its first particle
        int cell[3] = {0, 0, 0};
        if (have) {
            const int64_t i = VIA_PERM ? (int64_t)perm[jbeg] : jbeg;
#pragma unroll
            for (int c = 0; c < D; ++c) {
                T t = grid_coord(src.x[c][i], g.h[c], g.inv_h[c], g.hmul);
                cell[c] = cell_index(t, g.n[c]);
            }
        }
        // grid index of the nodes this lane stages and flushes: node t*GS + lg%GS of the stencil
        int noff[NPL];
#pragma unroll
        for (int t = 0; t < NPL; ++t) {
            const int node = t * GS + (lg % GS);
            const int ii = node % S, jj = (node / S) % S, kk = node / (S * S);
            const int sh = (S == 4) ? 1 : 0;
            const int gx = fold(cell[0] - sh + ii, g.n[0]), gy = fold(cell[1] - sh + jj, g.n[1]);
            const int gz = (D == 3) ? fold(cell[2] - sh + kk, g.n[2]) : 0;
            noff[t] = gx + g.n[0] * (gy + g.n[1] * gz);
        }

        // stage the field stencil of the cell in the group's shared-memory slot
        if constexpr (PUSH) {
            __syncwarp();
            if (have) {
#pragma unroll
                for (int c = 0; c < D; ++c)
#pragma unroll
                    for (int t = 0; t < NPL; ++t) s_E[gid][c][t * GS + (lg % GS)] = __ldg(f.E[c] + noff[t]);
            }
            __syncwarp();
        }

        T acc[DEP ? NODES : 1];
#pragma unroll
        for (int a = 0; a < (DEP ? NODES : 1); ++a) acc[a] = (T)0;

        // number of batches: warp-uniform
        int nb = (len + G * NB - 1) / (G * NB);
#pragma unroll
        for (int o = 16; o >= G; o >>= 1) nb = max(nb, __shfl_xor_sync(FULL, nb, o));

        for (int bt = 0; bt < nb; ++bt) {
            T wx[NB][S], wy[NB][S], wz[NB][S];
            T q[NB], xs[NB][D], vs[NB][D], wraw[NB];
            int64_t jp[NB];
            bool live[NB];
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const int k = (bt * NB + b) * G + lg;
                const bool in_item = k < len;
                jp[b] = jbeg + k;
                bool same = false;
                wraw[b] = (T)0;
                if (in_item) {
                    const int64_t i = VIA_PERM ? (int64_t)perm[jp[b]] : jp[b];
#pragma unroll
                    for (int c = 0; c < D; ++c) xs[b][c] = src.x[c][i];
                    if constexpr (PUSH) {
#pragma unroll
                        for (int c = 0; c < D; ++c) vs[b][c] = src.v[c][i];
                    }
                    if constexpr (DEP || VIA_PERM) wraw[b] = src.w[i];
                    same = cell_weights<T, P>(xs[b][0], g.h[0], g.inv_h[0], g.hmul, g.n[0], wx[b]) == cell[0];
                    same = (cell_weights<T, P>(xs[b][1], g.h[1], g.inv_h[1], g.hmul, g.n[1], wy[b]) == cell[1]) && same;
                    if constexpr (D == 3)
                        same = (cell_weights<T, P>(xs[b][D - 1], g.h[D - 1], g.inv_h[D - 1], g.hmul, g.n[D - 1], wz[b]) == cell[2]) && same;
                    if (!same) lone_particle<T, D, P, MODE, VIA_PERM>(src, i, dst, jp[b], g, f, racc, dt, qmdt);
                }
                if (!same) {
#pragma unroll
                    for (int i = 0; i < S; ++i) { wx[b][i] = (T)0; wy[b][i] = (T)0; wz[b][i] = (T)0; }
#pragma unroll
                    for (int c = 0; c < D; ++c) { xs[b][c] = (T)0; vs[b][c] = (T)0; }
                }
                if constexpr (D == 2) wz[b][0] = (T)1;
                live[b] = same;
                q[b] = same ? wraw[b] * g.inv_vol : (T)0;
            }

            T ec[NB][D];
#pragma unroll
            for (int b = 0; b < NB; ++b)
#pragma unroll
                for (int c = 0; c < D; ++c) ec[b][c] = (T)0;

#pragma unroll
            for (int kk = 0; kk < SZ; ++kk) {
#pragma unroll
                for (int jj = 0; jj < S; ++jj) {
                    const int row = (kk * S + jj) * S;
                    T er[D][S];
                    if constexpr (PUSH) {
#pragma unroll
                        for (int c = 0; c < D; ++c) load_row<T, S>(&s_E[gid][c][row], er[c]);
                    }
#pragma unroll
                    for (int b = 0; b < NB; ++b) {
                        const T wyz = wz[b][kk] * wy[b][jj];
                        if constexpr (DEP) {
                            const T qw = q[b] * wyz;
#pragma unroll
                            for (int i = 0; i < S; ++i) acc[row + i] = fma(qw, wx[b][i], acc[row + i]);
                        }
                        if constexpr (PUSH) {
#pragma unroll
                            for (int c = 0; c < D; ++c) {
                                T rsum = wx[b][0] * er[c][0];
#pragma unroll
                                for (int i = 1; i < S; ++i) rsum = fma(wx[b][i], er[c][i], rsum);
                                ec[b][c] = fma(wyz, rsum, ec[b][c]);
                            }
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
                            const T v = vs[b][c] + qmdt * ec[b][c];
                            dst.v[c][jp[b]] = v;
                            dst.x[c][jp[b]] = wrap_periodic(xs[b][c] + dt * v, g.L[c], g.inv_L[c]);
                        }
                        if constexpr (VIA_PERM) dst.w[jp[b]] = wraw[b];
                    }
                }
            }
        }

        // ---- end of the item: combine the G lanes' sums, add the totals to the grid
        if constexpr (DEP) {
            bool owner;
            group_combine<T, NODES, G>(acc, lg, owner);
            if (have && owner) {
#pragma unroll
                for (int t = 0; t < NPL; ++t) atomicAdd(&racc[noff[t]], (double)acc[t]);
            }
        }
    }
    (void)GROUPS;
}

// dynamic shared memory of k_cells: the field stencils of all groups
template <typename T, int D, int P, int MODE, int G>
constexpr size_t cells_smem_bytes()
{
    constexpr int S = StencilW<P>::S;
    constexpr int NODES = (D == 3) ? S * S * S : S * S;
    return (MODE & kModePush) ? sizeof(T) * (kCellThreads / G) * D * NODES : 16;
}

// launch k_cells over n particles sorted by cell.  VIA_PERM: particle perm[j] of src -> slot j of dst;
// otherwise in place on dst (src is ignored).  racc = double accumulation grid of the deposit.
template <typename T, int D, int P, int MODE, int G, int NB, bool VIA_PERM>
inline int launch_cells(const pic_grid_t& g, const pic_particles_t& src, const pic_particles_t& dst,
                        const int32_t* perm, const int32_t* cell_offsets, const void* const E[3], double* racc,
                        double dt, double qm, cudaStream_t st)
{
    if (dst.n <= 0) return PIC_OK;
    FieldP<T> f;
    for (int c = 0; c < 3; ++c) f.E[c] = (E && c < D) ? (const T*)E[c] : nullptr;
    auto kern = k_cells<T, D, P, MODE, G, NB, VIA_PERM>;
    constexpr size_t smem = cells_smem_bytes<T, D, P, MODE, G>();
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return PIC_ERR_CUDA;
        attr_set = true;
    }
    const unsigned blocks = (unsigned)((dst.n + kBlockParticles - 1) / kBlockParticles);
    kern<<<blocks, kCellThreads, smem, st>>>(make_partp<T>(VIA_PERM ? src : dst), make_partp<T>(dst), perm,
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
