// pic_nodes.cu -- pic_deposit_nodes: the COLLISION-FREE deposit, "threads on splines" (setrho_splines, PAPER.md:202-204
// section 3.3.1 with bucket-sorted particles, Fig. 6; Fortran of App. B): the threads are
// associated with the GRID data.  Every node j looks at the particles of the cells whose stencils reach it and adds
// up their spline values itself, so no two threads ever write the same node: no atomics, no race
// ("we avoid race condition and synchronization is no more necessary").  The paper's cost count,
// (Nx+d)(Ny+d)(Nz+d) Np / Nbuckets, is smallest "for buckets containing just one grid cell": that is the case
// built here (particles sorted by cell, cell_offsets from pic_sort).
//
// What this path adds to the hot path's deposit (k_runs: thread-private sums + one global reduction per node and
// run, whose order of additions is whatever the hardware makes it) is a FIXED order of additions: node j adds the
// contributions of its particles one by one in ascending position of the sorted array, each contribution computed
// in double with individually rounded operations (no fused multiply-add).  rho is therefore bitwise reproducible from
// run to run and from launch shape to launch shape, and it is the particle-order double sum of the definition
// rho[j] = h^-d sum_i w_i prod_c W_p(x_ic/h_c - j_c), rounded once to the storage type.
//
//   k_offsets_check        cell_offsets walkable (off[0] = 0, off[C] = N, non-decreasing)?  else *bad = 1
//   k_deposit_nodes        one thread per node; nodes with many particles around them go on a list instead
//   k_deposit_nodes_dense  one warp per listed node: the lanes compute 32 contributions at a time, the additions
//                          stay in order (same value as the one-thread sum, bit for bit)
//   fallback               a particle found outside the cell its position in the array says (the offsets do not
//                          describe the order) sets *bad: rho is then recomputed by the any-order run kernel.
#include "pic_runs.cuh"

namespace pic {

constexpr int kCtrNodesBad = 20, kCtrNodesDense = 21;     // words of SortWs::counters used here
constexpr int kDenseVisits = 4096;                         // a node with more particles around it gets a warp

__global__ void __launch_bounds__(256) k_offsets_check(const int32_t* __restrict__ off, int C, int64_t n, uint32_t* __restrict__ bad)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k > C) return;
    const int32_t a = off[k];
    bool b = a < 0 || (int64_t)a > n;
    if (k == 0) b = b || a != 0;
    if (k == C) b = b || (int64_t)a != n;
    if (k < C) b = b || off[k + 1] < a;
    if (b) *bad = 1u;
}

// num / 6 correctly rounded, without the division routine: q = RN(num * RN(1/6)) is within an ulp of the quotient,
// r = num - 6 q is exact in one fused operation, and RN(q + r * RN(1/6)) is then the correctly rounded quotient
// (Markstein's correction step; 6 is exactly representable and RN(1/6) is the correctly rounded reciprocal).
__device__ __forceinline__ double div6_rn(double num)
{
    const double y = 1.0 / 6.0;                            // RN(1/6), folded at compile time
    const double q = __dmul_rn(num, y);
    const double r = __fma_rn(-6.0, q, num);
    return __fma_rn(r, y, q);
}

// 1-D weight of a particle on the node with stencil index a (0..P), every operation rounded on its own, in the
// order of the definition's polynomial forms (R1): p = 1 (1 - xi, xi); p = 2 with d = xi - (nearest node - i0);
// p = 3 ((1-xi)^3, 3 xi^3 - 6 xi^2 + 4, -3 xi^3 + 3 xi^2 + 3 xi + 1, xi^3) / 6.  Branch-free: the lanes of a warp are
// neighbouring nodes and hold different a.
template <int P>
__device__ __forceinline__ bool node_weight(double xi, int i0, int jn, int n, double& w)
{
    int first;
    double d = xi;
    if constexpr (P == 1) {
        first = i0;
    } else if constexpr (P == 2) {
        const bool up = xi >= 0.5;
        d = __dsub_rn(xi, up ? 1.0 : 0.0);
        first = i0 + (up ? 1 : 0) - 1;
    } else {
        first = i0 - 1;
    }
    int a = jn - first;                                  // first in [-2, n]: one fold either way
    a = a < 0 ? a + n : a;
    a = a >= n ? a - n : a;
    if constexpr (P == 1) {
        w = a == 0 ? __dsub_rn(1.0, xi) : xi;
    } else if constexpr (P == 2) {
        const double s = a == 0 ? __dsub_rn(0.5, d) : __dadd_rn(0.5, d);
        const double side = __dmul_rn(__dmul_rn(0.5, s), s), mid = __dsub_rn(0.75, __dmul_rn(d, d));
        w = a == 1 ? mid : side;
    } else {
        const double x2 = __dmul_rn(xi, xi), x3 = __dmul_rn(x2, xi);
        const double om = __dsub_rn(1.0, xi);
        const double n0 = __dmul_rn(__dmul_rn(om, om), om);
        const double n1 = __dadd_rn(__dsub_rn(__dmul_rn(3.0, x3), __dmul_rn(6.0, x2)), 4.0);
        const double n2 = __dadd_rn(__dadd_rn(__dadd_rn(__dmul_rn(-3.0, x3), __dmul_rn(3.0, x2)), __dmul_rn(3.0, xi)), 1.0);
        const double num = a == 0 ? n0 : (a == 1 ? n1 : (a == 2 ? n2 : x3));
        w = div6_rn(num);
    }
    return a <= P;                                       // else the particle's stencil does not reach this node
}

// contribution of particle i to node jn[]; cc[] = the cell the particle must be in (else *wrong)
template <typename T, int D, int P>
__device__ __forceinline__ bool node_contribution(const PartP<T>& p, const GridP<T>& g, int64_t i, const int (&jn)[3],
                                                  const int (&cc)[3], double inv_vol, double& val, bool& wrong)
{
    double prod = 1.0;
    bool touch = true;
#pragma unroll
    for (int c = 0; c < D; ++c) {
        const T t = grid_coord(p.x[c][i], g.h[c], g.inv_h[c], g.hmul);
        const int i0 = cell_index(t, g.n[c]);
        if (i0 != cc[c]) wrong = true;
        const double xi = __dsub_rn((double)t, (double)i0);
        double w = 0.0;
        touch = node_weight<P>(xi, i0, jn[c], g.n[c], w) && touch;
        prod = c == 0 ? w : __dmul_rn(prod, w);
    }
    if (!touch) return false;
    val = __dmul_rn(__dmul_rn((double)p.w[i], inv_vol), prod);
    return true;
}

// the cells of one dimension whose particles can reach node j: j-1, j (p = 1) or j-2 .. j+1 (p = 2, 3), folded into
// [0, n), in ASCENDING order and without repeats: cell number q of m = min(count, n).  A fold happens at one end
// at most: the cells folded down from beyond n-1 come first, those folded up from below 0 last.
template <int P>
struct NodeCells {
    int m, hi, lw, base, n;
    __device__ __forceinline__ NodeCells(int j, int n_) : n(n_)
    {
        constexpr int lo = (P == 1) ? -1 : -2, cnt = (P == 1) ? 2 : 4;
        if (n_ < cnt) {                                   // a grid smaller than the reach: every cell, once
            m = n_; hi = 0; lw = 0; base = 0;
        } else {
            m = cnt;
            hi = max(0, j + lo + cnt - n_);
            lw = max(0, -(j + lo));
            base = max(j + lo, 0);
        }
    }
    __device__ __forceinline__ int cell(int q) const
    {
        return q < hi ? q : (q < m - lw ? base + (q - hi) : n - lw + (q - (m - lw)));
    }
};

template <typename T, int D, int P>
__global__ void __launch_bounds__(128) k_deposit_nodes(PartP<T> p, GridP<T> g, const int32_t* __restrict__ off, int64_t C,
                                                       double inv_vol, T* __restrict__ rho, uint32_t* __restrict__ bad,
                                                       uint32_t* __restrict__ dense_count, uint32_t* __restrict__ dense_list)
{
    if (*bad) return;
    const int64_t node = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (node >= C) return;
    int jn[3];
    jn[0] = (int)(node % g.n[0]);
    jn[1] = (int)((node / g.n[0]) % g.n[1]);
    jn[2] = (D == 3) ? (int)(node / ((int64_t)g.n[0] * g.n[1])) : 0;
    const NodeCells<P> ncx(jn[0], g.n[0]), ncy(jn[1], g.n[1]), ncz(jn[2], (D == 3) ? g.n[2] : 1);
    const int mx = ncx.m, my = ncy.m, mz = (D == 3) ? ncz.m : 1;
    // how many particles sit around this node?
    int64_t visits = 0;
    for (int a = 0; a < mz; ++a)
        for (int b = 0; b < my; ++b)
            for (int c = 0; c < mx; ++c) {
                const int64_t cell = ncx.cell(c) + (int64_t)g.n[0] * (ncy.cell(b) + (int64_t)g.n[1] * ((D == 3) ? ncz.cell(a) : 0));
                visits += off[cell + 1] - off[cell];
            }
    if (visits > kDenseVisits) {                           // a warp takes it (k_deposit_nodes_dense)
        dense_list[atomicAdd(dense_count, 1u)] = (uint32_t)node;
        return;
    }
    double acc = 0.0;
    bool wrong = false;
    for (int a = 0; a < mz; ++a)                           // cells in ascending key = ascending position of their particles
        for (int b = 0; b < my; ++b)
            for (int c = 0; c < mx; ++c) {
                const int cc[3] = {ncx.cell(c), ncy.cell(b), (D == 3) ? ncz.cell(a) : 0};
                const int64_t cell = cc[0] + (int64_t)g.n[0] * (cc[1] + (int64_t)g.n[1] * cc[2]);
                const int64_t end = off[cell + 1];
                for (int64_t i = off[cell]; i < end; ++i) {
                    double v;
                    if (node_contribution<T, D, P>(p, g, i, jn, cc, inv_vol, v, wrong)) acc = __dadd_rn(acc, v);
                }
            }
    rho[node] = (T)acc;
    if (wrong) *bad = 1u;
}

template <typename T, int D, int P>
__global__ void __launch_bounds__(128) k_deposit_nodes_dense(PartP<T> p, GridP<T> g, const int32_t* __restrict__ off,
                                                             double inv_vol, T* __restrict__ rho, uint32_t* __restrict__ bad,
                                                             const uint32_t* __restrict__ dense_count,
                                                             const uint32_t* __restrict__ dense_list)
{
    if (*bad) return;
    constexpr unsigned FULL = 0xFFFFFFFFu;
    const int lane = threadIdx.x & 31;
    const uint32_t m = *dense_count;
    const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
    for (uint32_t q = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; q < m; q += warps) {
        const int64_t node = dense_list[q];
        int jn[3];
        jn[0] = (int)(node % g.n[0]);
        jn[1] = (int)((node / g.n[0]) % g.n[1]);
        jn[2] = (D == 3) ? (int)(node / ((int64_t)g.n[0] * g.n[1])) : 0;
        const NodeCells<P> ncx(jn[0], g.n[0]), ncy(jn[1], g.n[1]), ncz(jn[2], (D == 3) ? g.n[2] : 1);
        const int mx = ncx.m, my = ncy.m, mz = (D == 3) ? ncz.m : 1;
        double acc = 0.0;
        bool wrong = false;
        for (int a = 0; a < mz; ++a)
            for (int b = 0; b < my; ++b)
                for (int c = 0; c < mx; ++c) {
                    const int cc[3] = {ncx.cell(c), ncy.cell(b), (D == 3) ? ncz.cell(a) : 0};
                    const int64_t cell = cc[0] + (int64_t)g.n[0] * (cc[1] + (int64_t)g.n[1] * cc[2]);
                    const int64_t end = off[cell + 1];
                    for (int64_t i0 = off[cell]; i0 < end; i0 += 32) {
                        const int64_t i = i0 + lane;
                        double v = 0.0;
                        const bool touch = i < end && node_contribution<T, D, P>(p, g, i, jn, cc, inv_vol, v, wrong);
                        unsigned todo = __ballot_sync(FULL, touch);
                        while (todo) {                     // the additions stay in position order
                            const int l = __ffs(todo) - 1;
                            acc = __dadd_rn(acc, __shfl_sync(FULL, v, l));
                            todo &= todo - 1;
                        }
                    }
                }
        if (lane == 0) rho[node] = (T)acc;
        if (wrong) *bad = 1u;
    }
}

// rho[k] = (T) racc[k] if *gate == want
template <typename T>
__global__ void __launch_bounds__(256) k_round_rho_gated(const double* __restrict__ racc, T* __restrict__ rho, int64_t C,
                                                         const uint32_t* __restrict__ gate, uint32_t want)
{
    if (*gate != want) return;
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < C) rho[k] = (T)racc[k];
}

template <typename T, int D, int P>
static int nodes_impl(const pic_grid_t& g, const pic_particles_t& p, const int32_t* off, void* rho, const SortWs& ws, cudaStream_t st)
{
    int64_t C = 1;
    double inv_vol = 1.0;
    for (int c = 0; c < g.dim; ++c) { C *= g.n[c]; inv_vol /= g.h[c]; }
    uint32_t* bad = ws.counters + kCtrNodesBad;
    uint32_t* dense_count = ws.counters + kCtrNodesDense;
    PIC_CUDA_OK(cudaMemsetAsync(bad, 0, 2 * sizeof(uint32_t), st));
    k_offsets_check<<<(unsigned)((C + 1 + 255) / 256), 256, 0, st>>>(off, (int)C, p.n, bad);
    const PartP<T> pp = make_partp<T>(p);
    const GridP<T> gp = make_gridp<T>(g);
    k_deposit_nodes<T, D, P><<<(unsigned)((C + 127) / 128), 128, 0, st>>>(pp, gp, off, C, inv_vol, (T*)rho, bad, dense_count, ws.idx[0]);
    k_deposit_nodes_dense<T, D, P><<<(unsigned)(sm_count() * 16), 128, 0, st>>>(pp, gp, off, inv_vol, (T*)rho, bad, dense_count, ws.idx[0]);
    count_launch(3);
    // offsets that do not describe the order: the any-order run kernel, selected on the device
    PIC_CUDA_OK(cudaMemsetAsync(ws.racc, 0, sizeof(double) * (size_t)C, st));
    if (p.n > 0) {
        int rc = launch_runs<T, D, P, kModeDeposit, false>(g, p, p, nullptr, nullptr, ws.racc, 0.0, 0.0, st, bad, 1u);
        if (rc != PIC_OK) return rc;
    }
    k_round_rho_gated<T><<<(unsigned)((C + 255) / 256), 256, 0, st>>>(ws.racc, (T*)rho, C, bad, 1u);
    count_launch();
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

template <typename T, int D>
static int nodes_order(const pic_grid_t& g, const pic_particles_t& p, const int32_t* off, void* rho, const SortWs& ws, cudaStream_t st)
{
    switch (g.order) {
    case 1: return nodes_impl<T, D, 1>(g, p, off, rho, ws, st);
    case 2: return nodes_impl<T, D, 2>(g, p, off, rho, ws, st);
    default: return nodes_impl<T, D, 3>(g, p, off, rho, ws, st);
    }
}

int launch_deposit_nodes(const pic_grid_t& g, const pic_particles_t& p, const int32_t* cell_offsets, void* rho,
                         const SortWs& ws, cudaStream_t st)
{
    if (g.dtype == PIC_F32)
        return g.dim == 2 ? nodes_order<float, 2>(g, p, cell_offsets, rho, ws, st) : nodes_order<float, 3>(g, p, cell_offsets, rho, ws, st);
    return g.dim == 2 ? nodes_order<double, 2>(g, p, cell_offsets, rho, ws, st) : nodes_order<double, 3>(g, p, cell_offsets, rho, ws, st);
}

// ---------------------------------------------------------------------------------------------------------------------
// pic_deposit_replicated: "collision-free: threads on buckets with data replication" (section 3.3.3,
// Fig. 7): "replicate the grid data from global to local data and sort particles in buckets ... associating threads
// with buckets of particles.  This ensures that each thread does the charge assignment on its local grid thus preventing
// race condition.  Guard-cells ... provide temporary memory for data exchange ... In the first step, reduction can be
// applied to local temporary variables without atomics in global memory.  In the second step, threads are assigned to
// the grid and collect the data from the temporary variables in global memory."  One cell per bucket:
//   k_deposit_cells_private  one thread per cell: its particles in order, the S^d nodes of the cell's stencil (the local
//                            grid with its guard nodes) summed in registers in double, written to slab[cell][S^d]
//   k_assemble_nodes         one thread per node: the local-grid entries of the cells around it, in ascending cell order
// No atomic anywhere, fixed order everywhere: bitwise reproducible.  (The association differs from the particle-order sum
// of pic_deposit_nodes: sums per cell first.)  Wrong offsets are found on the device and answered by the any-order kernel.
template <typename T, int D, int P>
__global__ void __launch_bounds__(64) k_deposit_cells_private(PartP<T> p, GridP<T> g, const int32_t* __restrict__ off, int64_t C,
                                                              double inv_vol, double* __restrict__ slab, uint32_t* __restrict__ bad)
{
    if (*bad) return;
    constexpr int S = StencilW<P>::S, SZ = (D == 3) ? S : 1;
    const int64_t cell = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= C) return;
    int cc[3];
    cc[0] = (int)(cell % g.n[0]);
    cc[1] = (int)((cell / g.n[0]) % g.n[1]);
    cc[2] = (D == 3) ? (int)(cell / ((int64_t)g.n[0] * g.n[1])) : 0;
    double acc[SZ][S][S];
#pragma unroll
    for (int a = 0; a < SZ; ++a)
#pragma unroll
        for (int b = 0; b < S; ++b)
#pragma unroll
            for (int c = 0; c < S; ++c) acc[a][b][c] = 0.0;
    bool wrong = false;
    const int32_t end = off[cell + 1];
    for (int32_t i = off[cell]; i < end; ++i) {
        double w[3][S];
#pragma unroll
        for (int c = 0; c < D; ++c) {
            T wt[S];
            const int i0 = cell_weights<T, P>(p.x[c][i], g.h[c], g.inv_h[c], g.hmul, g.n[c], wt);
            if (i0 != cc[c]) wrong = true;
#pragma unroll
            for (int a = 0; a < S; ++a) w[c][a] = (double)wt[a];
        }
        const double q = (double)p.w[i] * inv_vol;
#pragma unroll
        for (int a = 0; a < SZ; ++a) {
            const double qz = (D == 3) ? q * w[2][a] : q;
#pragma unroll
            for (int b = 0; b < S; ++b) {
                const double qy = qz * w[1][b];
#pragma unroll
                for (int c = 0; c < S; ++c) acc[a][b][c] = fma(qy, w[0][c], acc[a][b][c]);
            }
        }
    }
    double* mine = slab + cell * (int64_t)(SZ * S * S);
#pragma unroll
    for (int a = 0; a < SZ; ++a)
#pragma unroll
        for (int b = 0; b < S; ++b)
#pragma unroll
            for (int c = 0; c < S; ++c) mine[(a * S + b) * S + c] = acc[a][b][c];
    if (wrong) *bad = 1u;
}

// (cell, local index) pairs of one dimension whose local grid holds node j, ascending by cell then by index; at most 2 S
template <int P>
__device__ __forceinline__ int node_sources(int j, int n, int (&cell)[8], int (&loc)[8])
{
    constexpr int S = StencilW<P>::S, sh = (S == 4) ? 1 : 0;
    const NodeCells<P> nc(j, n);
    int m = 0;
    for (int q = 0; q < nc.m; ++q) {
        const int c = nc.cell(q);
        for (int a = 0; a < S; ++a)
            if (fold(c - sh + a, n) == j && m < 8) { cell[m] = c; loc[m] = a; ++m; }
    }
    return m;
}

template <typename T, int D, int P>
__global__ void __launch_bounds__(128) k_assemble_nodes(GridP<T> g, int64_t C, const double* __restrict__ slab, T* __restrict__ rho,
                                                        const uint32_t* __restrict__ bad)
{
    if (*bad) return;
    constexpr int S = StencilW<P>::S, SZ = (D == 3) ? S : 1;
    const int64_t node = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (node >= C) return;
    const int jx = (int)(node % g.n[0]), jy = (int)((node / g.n[0]) % g.n[1]);
    const int jz = (D == 3) ? (int)(node / ((int64_t)g.n[0] * g.n[1])) : 0;
    int cx[8], ax[8], cy[8], ay[8], cz[8] = {0, 0, 0, 0, 0, 0, 0, 0}, az[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    const int mx = node_sources<P>(jx, g.n[0], cx, ax), my = node_sources<P>(jy, g.n[1], cy, ay);
    const int mz = (D == 3) ? node_sources<P>(jz, g.n[2], cz, az) : 1;
    double acc = 0.0;
    for (int a = 0; a < mz; ++a)
        for (int b = 0; b < my; ++b)
            for (int c = 0; c < mx; ++c) {
                const int64_t cell = cx[c] + (int64_t)g.n[0] * (cy[b] + (int64_t)g.n[1] * cz[a]);
                acc += slab[cell * (int64_t)(SZ * S * S) + (az[a] * S + ay[b]) * S + ax[c]];
            }
    rho[node] = (T)acc;
}

size_t replicated_slab_bytes(const pic_grid_t& g)
{
    size_t C = 1, per = 1;
    const int S = g.order == 1 ? 2 : 4;
    for (int c = 0; c < g.dim; ++c) { C *= (size_t)g.n[c]; per *= (size_t)S; }
    return (C * per * sizeof(double) + 255) & ~(size_t)255;
}

template <typename T, int D, int P>
static int replicated_impl(const pic_grid_t& g, const pic_particles_t& p, const int32_t* off, void* rho, const SortWs& ws,
                           double* slab, cudaStream_t st)
{
    int64_t C = 1;
    double inv_vol = 1.0;
    for (int c = 0; c < g.dim; ++c) { C *= g.n[c]; inv_vol /= g.h[c]; }
    uint32_t* bad = ws.counters + kCtrNodesBad;
    PIC_CUDA_OK(cudaMemsetAsync(bad, 0, 2 * sizeof(uint32_t), st));
    k_offsets_check<<<(unsigned)((C + 1 + 255) / 256), 256, 0, st>>>(off, (int)C, p.n, bad);
    const GridP<T> gp = make_gridp<T>(g);
    k_deposit_cells_private<T, D, P><<<(unsigned)((C + 63) / 64), 64, 0, st>>>(make_partp<T>(p), gp, off, C, inv_vol, slab, bad);
    k_assemble_nodes<T, D, P><<<(unsigned)((C + 127) / 128), 128, 0, st>>>(gp, C, slab, (T*)rho, bad);
    count_launch(3);
    PIC_CUDA_OK(cudaMemsetAsync(ws.racc, 0, sizeof(double) * (size_t)C, st));
    if (p.n > 0) {
        int rc = launch_runs<T, D, P, kModeDeposit, false>(g, p, p, nullptr, nullptr, ws.racc, 0.0, 0.0, st, bad, 1u);
        if (rc != PIC_OK) return rc;
    }
    k_round_rho_gated<T><<<(unsigned)((C + 255) / 256), 256, 0, st>>>(ws.racc, (T*)rho, C, bad, 1u);
    count_launch();
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

template <typename T, int D>
static int replicated_order(const pic_grid_t& g, const pic_particles_t& p, const int32_t* off, void* rho, const SortWs& ws,
                            double* slab, cudaStream_t st)
{
    switch (g.order) {
    case 1: return replicated_impl<T, D, 1>(g, p, off, rho, ws, slab, st);
    case 2: return replicated_impl<T, D, 2>(g, p, off, rho, ws, slab, st);
    default: return replicated_impl<T, D, 3>(g, p, off, rho, ws, slab, st);
    }
}

int launch_deposit_replicated(const pic_grid_t& g, const pic_particles_t& p, const int32_t* cell_offsets, void* rho,
                              const SortWs& ws, void* slab, cudaStream_t st)
{
    if (g.dtype == PIC_F32)
        return g.dim == 2 ? replicated_order<float, 2>(g, p, cell_offsets, rho, ws, (double*)slab, st)
                          : replicated_order<float, 3>(g, p, cell_offsets, rho, ws, (double*)slab, st);
    return g.dim == 2 ? replicated_order<double, 2>(g, p, cell_offsets, rho, ws, (double*)slab, st)
                      : replicated_order<double, 3>(g, p, cell_offsets, rho, ws, (double*)slab, st);
}

}  // namespace pic
