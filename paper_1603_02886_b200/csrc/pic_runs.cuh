// pic_runs.cuh -- the kernel for particles grouped by cell: A WARP WALKS RUNS OF EQUAL CELL KEY.
//
// Deposit and/or gather+accel+push over particles in (mostly) cell order (rows a5-a7, fused a8,
// optionally with the reorder a4 through perm).  Prior art: the paper's CUDA kernel stages a
// per-block tile of rho in shared memory and atomicAdds every particle's 8 products into it
// ("sorting is required"); it also names reducing "on a temporary
// thread-private variable" and the collision-free "threads on splines" idea
// (setrho 3.3.1).  On sm_100a a floating-point atomicAdd on shared memory is a
// compare-and-swap loop, so the last two are what is built here, inside a warp:
//
//   * a warp owns WR consecutive slots of the order and takes them 32 at a time.
//     Phase W, lane = slot: coalesced loads (through perm when the reorder is fused in; the next
//     batch is prefetched), cell index, 1-D spline weights, one weight record per particle in shared
//     memory.  The cell KEY of every slot is compared with its left neighbour's: the batch falls into
//     RUNS of equal key.  Nothing else says where a cell starts -- cell_offsets is not read, so the
//     kernel is exact for ANY order (sorted input: one run per cell; stale order: shorter runs).
//   * Phase N, lanes on stencil rows: the warp holds ONE current cell.  Its S^d stencil nodes are
//     spread over G lanes (RPL rows of S x-neighbouring nodes each), replicated in the 32/G lane
//     groups: each lane keeps the d field components on its rows (the read-only
//     path, staged once per cell through shared memory) and its partial rho sums in registers.  The
//     groups take consecutive particles of the run, one each: read the record (broadcast loads),
//     form P = wz*wy*wx on the lane's rows, add q*P to the rho sums and P*E to the particle's
//     partial field (packed fma.rn.f32x2 on pairs of x-neighbouring nodes), and leave the partial
//     field in shared memory.
//   * Phase P, lane = slot again: sum the G partial fields, accel, push, wrap, coalesced stores.
//   * when the key changes (and every kFlushEvery particles of a long run, so that fp32 sums stay
//     short) the node sums of the groups are added up through shared memory and each node goes to
//     the grid with ONE global reduction (RED) in double precision.
//
// Registers hold RPL*S*(d+1) stencil values per lane; shared memory holds the records, the partial
// fields and the combine buffer (5 KB per warp for fp32 cubic 3-D).  No block-level barrier: warps
// are independent.
#pragma once
#include "pic_stencil.cuh"

namespace pic {

#ifndef PIC_RUNS_G32
#define PIC_RUNS_G32 4          // lanes per stencil, fp32
#endif
#ifndef PIC_RUNS_G64
#define PIC_RUNS_G64 8          // lanes per stencil, fp64
#endif
#ifndef PIC_RUNS_MINW32
#define PIC_RUNS_MINW32 14      // launch bound of the fp32 kernels (128 registers, 16 resident warps either way; 14 schedules 3 % faster than 13, 15, 16)
#endif
#ifndef PIC_RUNS_MINW64
#define PIC_RUNS_MINW64 10
#endif
#ifndef PIC_RUNS_WR
#define PIC_RUNS_WR 2048        // slots per warp
#endif
#ifndef PIC_RUNS_UNROLL
#define PIC_RUNS_UNROLL 2       // units of phase N in flight
#endif
#ifndef PIC_RUNS_WARPS
#define PIC_RUNS_WARPS 1        // warps per block (warps are independent)
#endif
#ifndef PIC_RUNS_BATCH_UNROLL
#define PIC_RUNS_BATCH_UNROLL 1   // batches of 32 slots per trip of the outer loop
#endif
constexpr int kRunsBatchUnroll = PIC_RUNS_BATCH_UNROLL;
constexpr int kRunsWarps = PIC_RUNS_WARPS;
constexpr int kRunsUnroll = PIC_RUNS_UNROLL;
constexpr int kRunsThreads = 32 * kRunsWarps;

template <typename T, int D, int P, int G_>
struct RunsShape {
    static constexpr int S = StencilW<P>::S;
    static constexpr int SZ = (D == 3) ? S : 1;
    static constexpr int ROWS = S * SZ;
    static constexpr int G = ROWS < G_ ? ROWS : G_;              // lanes per stencil
    static constexpr int RPL = ROWS / G;                         // rows per lane (consecutive, same z)
    static constexpr int NG = 32 / G;                            // groups = particles in flight
    static constexpr int NV = RPL * S;                           // node values per lane
    static constexpr int NODES = ROWS * S;                       // S^d
    static constexpr int NPL = (NODES + 31) / 32;                // stencil positions a lane fetches and flushes
    static constexpr int WR = PIC_RUNS_WR;
    static constexpr int RECW = D * S;                           // wx[S] wy[S] (wz[S])
    // strides of the per-particle rows in shared memory: an ODD number of 16-byte units, so that the 32 lanes of a
    // 128-bit access (lane = particle) spread over all banks (fp64 rows of 96 and 192 bytes hit 4 and 2 of the 8
    // 16-byte columns: half of that kernel's shared-memory wavefronts were bank conflicts)
    static constexpr int EPU = 16 / (int)sizeof(T);              // elements per 16-byte unit
    static constexpr int RECS = (((RECW + EPU - 1) / EPU) | 1) * EPU;      // weight record
    static constexpr int PARTS = (((D * G + EPU - 1) / EPU) | 1) * EPU;    // partial fields of one particle: [D][G]
    static constexpr int kFlushEvery = sizeof(T) == 4 ? 128 * NG : (1 << 30);
    // shared memory of one warp, in elements of T
    static constexpr int oRec = 0;                               // [32][RECS] weight records of the batch
    static constexpr int oQ = oRec + 32 * RECS;                  // [32] w / prod h
    static constexpr int oPart = oQ + 32;                        // [32][PARTS] partial fields
    static constexpr int oBuf = oPart + 32 * PARTS;              // [NG][NODES] node sums / [D][NODES] field of a cell
    static constexpr int nBuf = NG * NODES > D * NODES ? NG * NODES : D * NODES;
    static constexpr int oCol = oBuf + nBuf;                     // [D][ROWS] field on one node column
    static constexpr int warp_elems = (oCol + D * ROWS + 3) / 4 * 4;
    static constexpr size_t warp_bytes = sizeof(T) * warp_elems;
    static constexpr size_t bytes = warp_bytes * kRunsWarps;
    static_assert(RPL >= 1 && RPL <= S, "a lane's rows must share one z plane");
    static_assert(S % RPL == 0, "a lane's rows must not straddle z planes");
    static_assert(32 % S == 0 && (S & (S - 1)) == 0, "column slots are taken modulo S");
};

template <typename T>
constexpr int runs_min_blocks()
{
    return (sizeof(T) == 4 ? PIC_RUNS_MINW32 : PIC_RUNS_MINW64) / PIC_RUNS_WARPS;
}
// register budget of k_runs: a cap per thread (fp32: 136 registers = 15 warps per SM; at 128 ptxas spills a
// prefetched particle attribute, which exposes the whole memory latency), else a resident-block target
#ifdef PIC_RUNS_MAXREG32
#define PIC_RUNS_BOUNDS(T) __maxnreg__(sizeof(T) == 4 ? PIC_RUNS_MAXREG32 : 255)
#else
#define PIC_RUNS_BOUNDS(T) __launch_bounds__(kRunsThreads, (runs_min_blocks<T>()))
#endif

// v[s] <- v[(s - rho) mod S]: the weight of stencil column i goes to column slot (i + rho) mod S
template <typename T, int S>
__device__ __forceinline__ void rotate_slots(T (&v)[S], int rho)
{
    if constexpr (S == 4) {
        const bool r2 = (rho & 2) != 0, r1 = (rho & 1) != 0;
        const T a0 = r2 ? v[2] : v[0], a1 = r2 ? v[3] : v[1], a2 = r2 ? v[0] : v[2], a3 = r2 ? v[1] : v[3];
        v[0] = r1 ? a3 : a0; v[1] = r1 ? a0 : a1; v[2] = r1 ? a1 : a2; v[3] = r1 ? a2 : a3;
    } else {
        const bool r1 = (rho & 1) != 0;
        const T a0 = v[0], a1 = v[1];
        v[0] = r1 ? a1 : a0; v[1] = r1 ? a0 : a1;
    }
}

// The STRAYS k_runs has set aside (particles whose key differs from both neighbours': drifted particles of a
// stale order, one-particle cells), one thread each: "threads on particles" with global reductions (setrho
// 3.3.4; accel through the read-only path).  list[0 .. *count) holds their slots
// in p, where k_runs has left them un-advanced.
template <typename T, int D, int P, int MODE>
__global__ void __launch_bounds__(128) k_strays(PartP<T> p, GridP<T> g, FieldP<T> f, const uint32_t* __restrict__ list,
                                                const uint32_t* __restrict__ count, double* __restrict__ racc, double dtd, double qmdtd)
{
    const T dt = (T)dtd, qmdt = (T)qmdtd;
    const uint32_t m = *count;
    for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < m; t += gridDim.x * blockDim.x) {
        const uint32_t j = list[t];
        T x[D], v[D], e[D];
        int first[3] = {0, 0, 0};
        T wt[3][P + 1];
#pragma unroll
        for (int c = 0; c < D; ++c) {
            x[c] = p.x[c][j];
            e[c] = (T)0;
            const T tt = grid_coord(x[c], g.h[c], g.inv_h[c], g.hmul);
            spline_weights<T, P>(tt, cell_index(tt, g.n[c]), first[c], wt[c]);
        }
        const T q = (MODE & kModeDeposit) ? p.w[j] * g.inv_vol : (T)0;
        constexpr int PZ = (D == 3) ? P : 0;
#pragma unroll
        for (int cz = 0; cz <= PZ; ++cz) {
            const int jz = (D == 3) ? fold(first[2] + cz, g.n[2]) : 0;
            const T wz = (D == 3) ? wt[2][cz] : (T)1;
#pragma unroll
            for (int b = 0; b <= P; ++b) {
                const int jy = fold(first[1] + b, g.n[1]);
                const T wyz = wz * wt[1][b];
                const int row = g.n[0] * (jy + g.n[1] * jz);
#pragma unroll
                for (int a = 0; a <= P; ++a) {
                    const int at = row + fold(first[0] + a, g.n[0]);
                    const T wgt = wyz * wt[0][a];
                    if constexpr ((MODE & kModeDeposit) != 0) atomicAdd(&racc[at], (double)(q * wgt));
                    if constexpr ((MODE & kModePush) != 0) {
#pragma unroll
                        for (int c = 0; c < D; ++c) e[c] += wgt * __ldg(f.E[c] + at);
                    }
                }
            }
        }
        if constexpr ((MODE & kModePush) != 0) {
#pragma unroll
            for (int c = 0; c < D; ++c) {
                const T v0 = p.v[c][j];
                v[c] = v0 + qmdt * e[c];
                T xn = x[c] + dt * v[c];
                if (!(xn >= (T)0 && xn < g.L[c])) xn = advance_wrap<T>(x[c], v0, e[c], dtd, qmdtd, g.Ld[c]);
                p.v[c][j] = v[c];
                p.x[c][j] = xn;
            }
        }
    }
}

// STRAYS: lone particles are set aside in stray_list for k_strays (used where the order may be stale)
// EMIT:   the next sort's inputs are written as the particles are pushed (sorted input only: !STRAYS)
// HM:     every spacing is a power of two, so x/h is the product x * (1/h) bit for bit (R13): no division path
template <typename T, int D, int P, int MODE, bool VIA_PERM, int G_, bool STRAYS, bool EMIT, bool HM>
__global__ void PIC_RUNS_BOUNDS(T)
k_runs(PartP<T> src, PartP<T> dst, const int32_t* __restrict__ perm, GridP<T> g, FieldP<T> f, int64_t n,
       double* __restrict__ racc, double dtd, double qmdtd, const uint32_t* __restrict__ gate, uint32_t want,
       uint32_t* __restrict__ stray_list, uint32_t* __restrict__ stray_count, EmitP em)
{
    static_assert(!EMIT || (!STRAYS && (MODE & kModePush) != 0), "emission needs the push and exact cell order");
    static_assert(!EMIT || PIC_RUNS_WR == kStageTile, "one warp's range is one staging tile");
    using SH = RunsShape<T, D, P, G_>;
    if (gate && *gate != want) return;                // the other arm of a device-side choice runs instead
    const T dt = (T)dtd, qmdt = (T)qmdtd;
    const int hm = HM ? 1 : g.hmul;
    constexpr int S = SH::S, S2 = S / 2, SZ = SH::SZ, ROWS = SH::ROWS;
    constexpr int G = SH::G, RPL = SH::RPL, NG = SH::NG, NV = SH::NV, NODES = SH::NODES, NPL = SH::NPL;
    constexpr int WR = SH::WR, RECS = SH::RECS, PARTS = SH::PARTS;
    constexpr bool DEP = (MODE & kModeDeposit) != 0, PUSH = (MODE & kModePush) != 0;
    constexpr unsigned FULL = 0xFFFFFFFFu;
    constexpr int sh = (S == 4) ? 1 : 0;              // the cell's stencil starts at node column cx - sh
    constexpr uint32_t B = sizeof(T);

    extern __shared__ __align__(16) unsigned char s_dyn[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int lg = lane % G, grp = lane / G;
    const uint32_t sb = smem_base(s_dyn) + (uint32_t)(warp * SH::warp_bytes);
    const uint32_t a_rec = sb + SH::oRec * B, a_q = sb + SH::oQ * B, a_part = sb + SH::oPart * B;
    const uint32_t a_buf = sb + SH::oBuf * B, a_col = sb + SH::oCol * B;

    const int64_t j0 = ((int64_t)blockIdx.x * kRunsWarps + warp) * WR;
    if (j0 >= n) return;                              // warps are independent: no block barrier below
    const int cnt = (int)((n - j0 < (int64_t)WR) ? (n - j0) : (int64_t)WR);

    // rows of this lane: r = lg*RPL + rr: z plane kk, y rows jj0 .. jj0+RPL-1
    const int kk = (lg * RPL) / S, jj0 = (lg * RPL) % S;

    // ---- the current cell (warp-uniform) and this lane's share of its stencil.  Node COLUMNS live in slots:
    //      column u (unfolded x index) is held in slot u mod S, so that the step to the x-neighbour cell
    //      replaces ONE column and leaves the other S-1 where they are.
    int cur = -1, ccx = 0, ccy = 0, ccz = 0;
    int since = 0;                                    // particles added to the node sums since the last full flush
    Pk<T> Er[PUSH ? D : 1][RPL][S2];                  // field on (row, slot pair)
    Pk<T> acc[DEP ? RPL : 1][S2];                     // rho sums on (row, slot pair)
#pragma unroll
    for (int rr = 0; rr < (DEP ? RPL : 1); ++rr)
#pragma unroll
        for (int i = 0; i < S2; ++i) acc[rr][i] = pk_zero<T>();
    int nidx[NPL];                                    // grid index of stencil position lane + 32 m = row*S + slot
    int rowb = 0;                                     // grid index of (x = 0, row lane mod ROWS)
#pragma unroll
    for (int m = 0; m < NPL; ++m) nidx[m] = 0;

    // all node sums -> one global reduction per node ("only once with atomic adds")
    auto flush_all = [&]() {
        const uint32_t mine = a_buf + (uint32_t)(grp * NODES + lg * NV) * B;
#pragma unroll
        for (int rr = 0; rr < RPL; ++rr) {
            T a[S];
#pragma unroll
            for (int i = 0; i < S2; ++i) { a[2 * i] = pk_lo(acc[rr][i]); a[2 * i + 1] = pk_hi(acc[rr][i]); acc[rr][i] = pk_zero<T>(); }
            sts<T, S>(mine + rr * S * B, a);
        }
        __syncwarp();
#pragma unroll
        for (int m = 0; m < NPL; ++m) {
            const int nid = lane + 32 * m;
            if (NODES % 32 == 0 || nid < NODES) {
                T s = lds1<T>(a_buf + (uint32_t)nid * B);
#pragma unroll
                for (int q = 1; q < NG; ++q) s += lds1<T>(a_buf + (uint32_t)(q * NODES + nid) * B);
                if (s != (T)0) atomicAdd(&racc[nidx[m]], (double)s);
            }
        }
        __syncwarp();
        since = 0;
    };
    // a new cell anywhere: every column is flushed and fetched
    auto jump_to = [&](int nx_, int ny_, int nz_) {
        int nnew[NPL];
        const int rho = (nx_ - sh) & (S - 1);
#pragma unroll
        for (int m = 0; m < NPL; ++m) {
            const int nid = lane + 32 * m;
            const int s = nid % S, r = nid / S, jy = r % S, kz = (r / S) % SZ;    // lanes beyond NODES: any valid node
            const int i = (s - rho) & (S - 1);
            const int gx = fold(nx_ - sh + i, g.n[0]);
            const int gy = fold(ny_ - sh + jy, g.n[1]);
            const int gz = (D == 3) ? fold(nz_ - sh + kz, g.n[2]) : 0;
            nnew[m] = gx + g.n[0] * (gy + g.n[1] * gz);
        }
        if (DEP && since > 0) flush_all();
#pragma unroll
        for (int m = 0; m < NPL; ++m) nidx[m] = nnew[m];
        {
            const int r = lane % ROWS, jy = r % S, kz = r / S;
            const int gy = fold(ny_ - sh + jy, g.n[1]);
            const int gz = (D == 3) ? fold(nz_ - sh + kz, g.n[2]) : 0;
            rowb = g.n[0] * (gy + g.n[1] * gz);
        }
        ccx = nx_; ccy = ny_; ccz = nz_;
        if constexpr (PUSH) {
            cp_async_wait();                          // (a column fetched ahead for the old row is dropped)
            if (lane < ROWS) {                        // the column the next slide will need
                const int xnext = fold(ccx - sh + S, g.n[0]);
#pragma unroll
                for (int c = 0; c < D; ++c) cp_async_elem(a_col + (uint32_t)(c * ROWS + lane) * B, f.E[c] + rowb + xnext);
            }
#pragma unroll
            for (int m = 0; m < NPL; ++m) {
                const int nid = lane + 32 * m;
                if (NODES % 32 == 0 || nid < NODES) {
#pragma unroll
                    for (int c = 0; c < D; ++c) sts1<T>(a_buf + (uint32_t)(c * NODES + nid) * B, ldg_here(f.E[c] + nidx[m]));
                }
            }
            __syncwarp();
#pragma unroll
            for (int c = 0; c < D; ++c)
#pragma unroll
                for (int rr = 0; rr < RPL; ++rr) {
                    T v[S];
                    lds<T, S>(a_buf + (uint32_t)(c * NODES + lg * NV + rr * S) * B, v);
#pragma unroll
                    for (int i = 0; i < S2; ++i) Er[c][rr][i] = pk_make(v[2 * i], v[2 * i + 1]);
                }
            __syncwarp();
        }
    };
    // the x-neighbour cell: column ccx - sh retires (its sums go to the grid), column ccx - sh + S takes its slot
    auto slide = [&]() {
        const int rho = (ccx - sh) & (S - 1);
        const int xold = fold(ccx - sh, g.n[0]), xnew = fold(ccx - sh + S, g.n[0]);
        const bool rown = lane < ROWS;
        if (DEP && since > 0) {
            T col[RPL];
#pragma unroll
            for (int s = 0; s < S; ++s)
                if (rho == s) {                       // warp-uniform
#pragma unroll
                    for (int rr = 0; rr < RPL; ++rr) {
                        const Pk<T> a = acc[rr][s / 2];
                        col[rr] = (s & 1) ? pk_hi(a) : pk_lo(a);
                        acc[rr][s / 2] = (s & 1) ? pk_make(pk_lo(a), (T)0) : pk_make((T)0, pk_hi(a));
                    }
                }
            sts<T, RPL>(a_buf + (uint32_t)(grp * ROWS + lg * RPL) * B, col);
            __syncwarp();
            if (rown) {
                T s = lds1<T>(a_buf + (uint32_t)lane * B);
#pragma unroll
                for (int q = 1; q < NG; ++q) s += lds1<T>(a_buf + (uint32_t)(q * ROWS + lane) * B);
                if (s != (T)0) atomicAdd(&racc[rowb + xold], (double)s);
            }
        }
        if constexpr (PUSH) {
            cp_async_wait();                          // the column was fetched ahead, see below and jump_to
        }
        __syncwarp();
        if constexpr (PUSH) {
#pragma unroll
            for (int c = 0; c < D; ++c) {
                T v[RPL];
                lds<T, RPL>(a_col + (uint32_t)(c * ROWS + lg * RPL) * B, v);
#pragma unroll
                for (int s = 0; s < S; ++s)
                    if (rho == s) {                   // warp-uniform
#pragma unroll
                        for (int rr = 0; rr < RPL; ++rr)
                            Er[c][rr][s / 2] = (s & 1) ? pk_make(pk_lo(Er[c][rr][s / 2]), v[rr]) : pk_make(v[rr], pk_hi(Er[c][rr][s / 2]));
                    }
            }
        }
        if ((lane & (S - 1)) == rho) {
#pragma unroll
            for (int m = 0; m < NPL; ++m) nidx[m] += xnew - xold;
        }
        ccx += 1;
        if constexpr (PUSH) {
            __syncwarp();                             // every lane has read the column: fetch the next one ahead
            if (rown) {
                const int xnext = fold(ccx - sh + S, g.n[0]);
#pragma unroll
                for (int c = 0; c < D; ++c) cp_async_elem(a_col + (uint32_t)(c * ROWS + lane) * B, f.E[c] + rowb + xnext);
            }
        }
    };

    // particle of this lane in the current batch, and the prefetched one of the next batch
    T nx[D], nv[D], nw = (T)0;
#pragma unroll
    for (int c = 0; c < D; ++c) { nx[c] = (T)0; nv[c] = (T)0; }
    int in1 = 0;                                      // source index of this lane's slot in batch b+1 (then b+2)
    uint32_t emitted = 0;                             // EMIT: movers of this warp's range so far
    auto load_attrs = [&](int i) {
#pragma unroll
        for (int c = 0; c < D; ++c) {
            nx[c] = src.x[c][i];
            if constexpr (PUSH || VIA_PERM) nv[c] = src.v[c][i];
        }
        if constexpr (DEP || VIA_PERM) nw = src.w[i];
    };
    const int64_t jl = j0 + lane;
    if (lane < cnt) {
        in1 = VIA_PERM ? perm[jl] : (int)jl;
        load_attrs(in1);
    }
    if (32 + lane < cnt) in1 = VIA_PERM ? perm[jl + 32] : (int)jl + 32;

#pragma unroll (kRunsBatchUnroll)
    for (int b0 = 0; b0 < cnt; b0 += 32) {
        const int nb = (cnt - b0 < 32) ? cnt - b0 : 32;
        const bool valid = lane < nb;
        T px[D], pv[D], pw = nw;
#pragma unroll
        for (int c = 0; c < D; ++c) { px[c] = nx[c]; pv[c] = nv[c]; }
        // prefetch: attributes of the next batch (index known), index of the one after
        if (b0 + 32 + lane < cnt) load_attrs(in1);
        if (b0 + 64 + lane < cnt) in1 = VIA_PERM ? perm[jl + b0 + 64] : (int)jl + b0 + 64;

        // ---- phase W: lane = slot
        int key = -1, c0, c1, c2 = 0;
        int idx = lane, nrec = nb;                    // this lane's record index, records in the batch
        bool lonely = false;
        auto write_record = [&]() {
            T w1[S], w2[S], w3[SZ];
            const int cx = cell_weights<T, P>(px[0], g.h[0], g.inv_h[0], hm, g.n[0], w1);
            const int cy = cell_weights<T, P>(px[1], g.h[1], g.inv_h[1], hm, g.n[1], w2);
            int cz = 0;
            if constexpr (D == 3) cz = cell_weights<T, P>(px[2], g.h[2], g.inv_h[2], hm, g.n[2], w3);
            if constexpr (!STRAYS) {
                c0 = cx; c1 = cy; c2 = cz;
                if (valid) key = c0 + g.n[0] * (c1 + g.n[1] * c2);
            }
            rotate_slots<T, S>(w1, cx - sh);          // x weights by column slot
            const uint32_t rec = a_rec + (uint32_t)(idx * RECS) * B;
            sts<T, S>(rec, w1);
            sts<T, S>(rec + S * B, w2);
            if constexpr (D == 3) sts<T, S>(rec + 2 * S * B, w3);
            if constexpr (DEP) sts1<T>(a_q + (uint32_t)idx * B, (valid && !lonely) ? pw * g.inv_vol : (T)0);
        };
        if constexpr (STRAYS) {
            c0 = cell_index(grid_coord(px[0], g.h[0], g.inv_h[0], hm), g.n[0]);
            c1 = cell_index(grid_coord(px[1], g.h[1], g.inv_h[1], hm), g.n[1]);
            if constexpr (D == 3) c2 = cell_index(grid_coord(px[2], g.h[2], g.inv_h[2], hm), g.n[2]);
            if (valid) key = c0 + g.n[0] * (c1 + g.n[1] * c2);
            // a particle whose key differs from both neighbours' is a STRAY: it does not break the run around it but
            // is set aside for k_strays.  The others are the RECORDS of the batch, in order.
            const int kleft = __shfl_up_sync(FULL, key, 1), kright = __shfl_down_sync(FULL, key, 1);
            lonely = valid && key != (lane == 0 ? cur : kleft) && (lane == nb - 1 || key != kright);
            const unsigned strays = __ballot_sync(FULL, lonely);
            if (strays) {                             // warp-uniform; rare in cell order: compact the records
                const unsigned keep = (nb == 32 ? FULL : ((1u << nb) - 1u)) & ~strays, below = (1u << lane) - 1u;
                nrec = __popc(keep);
                idx = lonely ? nrec + __popc(strays & below) : __popc(keep & below);  // (strays: unused records behind)
                uint32_t at = 0;
                if (lane == 0) at = atomicAdd(stray_count, (uint32_t)__popc(strays));
                at = __shfl_sync(FULL, at, 0);
                if (lonely) stray_list[at + __popc(strays & below)] = (uint32_t)(jl + b0);
                write_record();                       // (own cell: before the keys are permuted)
                const uint32_t tmp = a_part;          // the partial-field buffer is free here: 4 ints per record
                if (valid && !lonely)
                    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" :: "r"(tmp + idx * 16), "r"(key), "r"(c0), "r"(c1), "r"(c2) : "memory");
                __syncwarp();
                key = -1;
                if (lane < nrec)
                    asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(key), "=r"(c0), "=r"(c1), "=r"(c2) : "r"(tmp + lane * 16));
                __syncwarp();
            } else {
                write_record();
            }
        } else {
            write_record();
        }
        // key, c0, c1, c2 now belong to record `lane`
        const int kprev = __shfl_up_sync(FULL, key, 1);
        const unsigned heads = __ballot_sync(FULL, lane < nrec && key != (lane == 0 ? cur : kprev));
        __syncwarp();

        // ---- phase N: lanes on stencil rows, run by run
        int pos = 0;
        while (pos < nrec) {
            const bool head = (heads >> pos) & 1u;
            if (head) {                               // the key changes here
                const bool had = cur >= 0;
                cur = __shfl_sync(FULL, key, pos);
                const int nx_ = __shfl_sync(FULL, c0, pos), ny_ = __shfl_sync(FULL, c1, pos);
                const int nz_ = (D == 3) ? __shfl_sync(FULL, c2, pos) : 0;
                const int dx = nx_ - ccx;
                if (had && ny_ == ccy && nz_ == ccz && dx >= 1 && dx < S) {
                    for (int k = 0; k < dx; ++k) slide();         // same grid row, at most S-1 cells on
                } else {
                    jump_to(nx_, ny_, nz_);
                }
            } else if (DEP && since >= SH::kFlushEvery) {
                flush_all();
            }
            const unsigned above = (pos < 31) ? (heads & ~((2u << pos) - 1u)) : 0u;
            const int end = above ? __ffs(above) - 1 : nrec;
            // the groups take records pos.., one each; a group beyond the end repeats the last record with q = 0
#pragma unroll (STRAYS ? 1 : kRunsUnroll)
            for (int u = pos; u < end; u += NG) {
                const bool live = u + grp < end;
                const int r = live ? u + grp : end - 1;
                const uint32_t rp = a_rec + (uint32_t)(r * RECS) * B;
                T wyv[RPL];
                Pk<T> wx2[S2];
                lds_pairs<S2>(rp, wx2);
                lds<T, RPL>(rp + (uint32_t)(S + jj0) * B, wyv);
                const T wzv = (D == 3) ? lds1<T>(rp + (uint32_t)(2 * S + kk) * B) : (T)1;
                T qv = (T)0;
                if constexpr (DEP) { qv = lds1<T>(a_q + (uint32_t)r * B); qv = live ? qv : (T)0; }
                Pk<T> sum[PUSH ? D : 1];
                const Pk<T> q2 = pk_make(qv, qv);
                bool first = true;
#pragma unroll
                for (int rr = 0; rr < RPL; ++rr) {
                    const T a = wzv * wyv[rr];
                    const Pk<T> a2 = pk_make(a, a);
#pragma unroll
                    for (int i = 0; i < S2; ++i) {
                        const Pk<T> pp = pk_mul(a2, wx2[i]);
                        if constexpr (DEP) pk_acc(acc[rr][i], q2, pp);
                        if constexpr (PUSH) {
#pragma unroll
                            for (int c = 0; c < D; ++c) {
                                if (first) sum[c] = pk_mul(pp, Er[c][rr][i]);
                                else pk_acc(sum[c], pp, Er[c][rr][i]);
                            }
                        }
                        first = false;
                    }
                }
                if constexpr (PUSH) {                 // (a repeated record writes the same values again)
#pragma unroll
                    for (int c = 0; c < D; ++c)
                        sts1<T>(a_part + (uint32_t)(r * PARTS + c * G + lg) * B, pk_lo(sum[c]) + pk_hi(sum[c]));
                }
            }
            since += end - pos;
            pos = end;
        }
        __syncwarp();

        // ---- phase P: lane = slot again: accel + push + store
        if (valid) {
            const int64_t j = jl + b0;
            if (PUSH && !lonely) {
                bool inside = true;
                T e[D], vn[D], xn[D];
#pragma unroll
                for (int c = 0; c < D; ++c) {
                    T pe[G];
                    lds<T, G>(a_part + (uint32_t)(idx * PARTS + c * G) * B, pe);
                    e[c] = pe[0];
#pragma unroll
                    for (int q = 1; q < G; ++q) e[c] += pe[q];
                    vn[c] = pv[c] + qmdt * e[c];
                    xn[c] = px[c] + dt * vn[c];
                    inside = inside && (xn[c] >= (T)0 && xn[c] < g.L[c]);
                }
                if (!inside) {                        // one rare branch for all components
#pragma unroll
                    for (int c = 0; c < D; ++c) xn[c] = advance_wrap<T>(px[c], pv[c], e[c], dtd, qmdtd, g.Ld[c]);
                }
#pragma unroll
                for (int c = 0; c < D; ++c) { px[c] = xn[c]; pv[c] = vn[c]; }
            }
            if ((PUSH && !lonely) || VIA_PERM) {
#pragma unroll
                for (int c = 0; c < D; ++c) { dst.x[c][j] = px[c]; dst.v[c][j] = pv[c]; }
                if constexpr (VIA_PERM) dst.w[j] = pw;
            }
        }
        if constexpr (EMIT) {
            // next key of the advanced particle: the same function of the stored position that k_classify applies
            int nk = 0, mul = 1;
#pragma unroll
            for (int c = 0; c < D; ++c) {
                nk += mul * cell_index(grid_coord(px[c], g.h[c], g.inv_h[c], hm), g.n[c]);
                mul *= g.n[c];
            }
            const bool mover = valid && nk != key;
            const unsigned bal = __ballot_sync(FULL, mover);
            const uint32_t slot = (uint32_t)j0 + (uint32_t)(b0 + lane);   // N < 2^30: 32-bit slot numbers
            if (valid) em.pkey[slot] = (uint32_t)nk;
            if (mover) {
                const uint32_t at = (uint32_t)j0 + emitted + (uint32_t)__popc(bal & ((1u << lane) - 1u));
                em.stage_key[at] = (uint32_t)nk;
                em.stage_idx[at] = slot;
                // histograms: one particle fewer in the present cell, one mover more in the next one (the second
                // word counts those that come from below); the sort puts count = old count - out + in together
                atomicAdd(&em.cell_out[key], 1);
                atomicAdd(&em.mover_in[nk], (nk > key) ? 0x100000001ull : 1ull);
            }
            if (lane == 0) {
                const uint32_t word = ((uint32_t)j0 + (uint32_t)b0) >> 5;
                em.mask[word] = bal;
                em.mprefix[word] = emitted;
            }
            emitted += (uint32_t)__popc(bal);
        }
    }
    if constexpr (EMIT) {
        if (lane == 0) em.tile_count[j0 / WR] = (int32_t)emitted;
    }
    if (DEP && since > 0) flush_all();
    if constexpr (PUSH) cp_async_wait();              // a column fetched ahead may still be in flight
}

// launch k_runs over n particles.  VIA_PERM: particle perm[j] of src -> slot j of dst; otherwise in place
// on dst.  racc = double accumulation grid of the deposit.  The kernel runs only if *gate == want (gate
// may be NULL).  stray_list / stray_count (both or neither; *stray_count zeroed by the caller): lone particles
// are set aside there for launch_strays instead of breaking the run they sit in.  emit != NULL (MODE both, no
// strays): the next sort's inputs are written too.
template <typename T, int D, int P, int MODE, bool VIA_PERM>
inline int launch_runs(const pic_grid_t& g, const pic_particles_t& src, const pic_particles_t& dst,
                       const int32_t* perm, const void* const E[3], double* racc, double dt, double qm,
                       cudaStream_t st, const uint32_t* gate = nullptr, uint32_t want = 0,
                       uint32_t* stray_list = nullptr, uint32_t* stray_count = nullptr, const EmitP* emit = nullptr)
{
    if (dst.n <= 0) return PIC_OK;
    constexpr int GP = sizeof(T) == 4 ? PIC_RUNS_G32 : PIC_RUNS_G64;
    using SH = RunsShape<T, D, P, GP>;
    FieldP<T> f;
    for (int c = 0; c < 3; ++c) f.E[c] = (E && c < D) ? (const T*)E[c] : nullptr;
    constexpr size_t smem = SH::bytes;
    static_assert(smem <= 48 * 1024, "k_runs relies on the default dynamic shared memory limit");
    constexpr int64_t per_block = (int64_t)SH::WR * kRunsWarps;
    const unsigned blocks = (unsigned)((dst.n + per_block - 1) / per_block);
    const EmitP none{};
    const GridP<T> gp = make_gridp<T>(g);
    const PartP<T> ps = make_partp<T>(VIA_PERM ? src : dst), pd = make_partp<T>(dst);
    auto go = [&](auto kern, uint32_t* sl, uint32_t* sc, const EmitP& em) {
        kern<<<blocks, kRunsThreads, smem, st>>>(ps, pd, perm, gp, f, dst.n, racc, dt, qm * dt, gate, want, sl, sc, em);
        count_launch();
        return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
    };
    if constexpr (MODE == kModeBoth) {
        if (emit)
            return gp.hmul ? go(k_runs<T, D, P, MODE, VIA_PERM, GP, false, true, true>, nullptr, nullptr, *emit)
                           : go(k_runs<T, D, P, MODE, VIA_PERM, GP, false, true, false>, nullptr, nullptr, *emit);
    }
    if (stray_list && stray_count) return go(k_runs<T, D, P, MODE, VIA_PERM, GP, true, false, false>, stray_list, stray_count, none);
    return go(k_runs<T, D, P, MODE, VIA_PERM, GP, false, false, false>, nullptr, nullptr, none);
}

// the particles k_runs has set aside, in place on p
template <typename T, int D, int P, int MODE>
inline int launch_strays(const pic_grid_t& g, const pic_particles_t& p, const void* const E[3], double* racc, double dt,
                         double qm, const uint32_t* stray_list, const uint32_t* stray_count, int sms, cudaStream_t st)
{
    if (p.n <= 0) return PIC_OK;
    FieldP<T> f;
    for (int c = 0; c < 3; ++c) f.E[c] = (E && c < D) ? (const T*)E[c] : nullptr;
    k_strays<T, D, P, MODE><<<(unsigned)(sms * 8), 128, 0, st>>>(make_partp<T>(p), make_gridp<T>(g), f, stray_list, stray_count,
                                                              racc, dt, qm * dt);
    count_launch();
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

}  // namespace pic
