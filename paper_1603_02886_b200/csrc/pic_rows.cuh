// pic_rows.cuh -- the kernel for particles grouped by cell: LANES ON STENCIL ROWS.
//
// Deposit and/or gather+accel+push over particles sorted by cell (rows a5-a7, fused a8, optionally
// with the reorder a4 through perm).  Prior art: the paper's CUDA kernel stages a per-block tile of
// rho in shared memory and atomicAdds every particle's 8 products into it ("sorting is required",
// PAPER.md:294, 504-525); it also names reducing "on a temporary thread-private variable"
// (PAPER.md:300).  On sm_100a a floating-point atomicAdd on shared memory is a compare-and-swap
// loop, and S^d thread-private sums per particle lane cost 64 registers and a combine per cell
// (measured: slower).  Here the paper's other collision-free idea is applied INSIDE a
// cell: "threads on splines" (setrho 3.3.1) -- every lane owns grid nodes, not
// particles:
//
//   * a warp owns WR consecutive slots of the sorted order, lists the cell runs inside them
//     ("items", at most kItemMax particles, in cell order) and works through them NG = 32/G at a
//     time: a GROUP of G lanes per item.  No block-level barrier anywhere: warps are independent.
//   * lane lg of a group owns RPL = S^(d-1)/G rows of the cell's S^d stencil (a row = S
//     x-neighbouring nodes).  It keeps, in registers, the d field components on those rows
//     (loaded once per item with read-only loads) and the rho sums of those nodes.
//   * particles are taken G at a time.  Phase W (lane = particle): the lane reads its particle
//     straight from global memory (through perm when the reorder is fused in; the next batch is
//     prefetched into registers), computes the 1-D spline weights and writes them as one record
//     to the group's shared-memory scratch.  Phase N (lane = rows): every lane reads each of the G
//     records (broadcast loads), forms the products P = wz*wy*wx on its rows, adds q*P to its rho
//     sums and P*E to the particle's partial field.  A transposed butterfly of shuffles then hands
//     lane lg the total field of particle lg, which it accelerates, pushes and stores.
//   * at the end of the item each lane adds its RPL*S node sums to the grid with global
//     reductions (RED) in double precision.
//
// Shared memory holds only the weight records and the item list (9 KB per warp); registers hold
// RPL*S*(d+1) stencil values instead of S^d sums (fp32 cubic 3-D: 168 registers, 12 warps per SM).
#pragma once
#include "pic_stencil.cuh"

namespace pic {

#ifndef PIC_ROWS_G32
#define PIC_ROWS_G32 4          // lanes per item, fp32
#endif
#ifndef PIC_ROWS_MINW32
#define PIC_ROWS_MINW32 12      // resident warps per SM the fp32 kernels are compiled for (168 registers)
#endif
#ifndef PIC_ROWS_WR
#define PIC_ROWS_WR 1024
#endif
#ifndef PIC_ROWS_WARPS
#define PIC_ROWS_WARPS 1        // warps per block (warps are independent; one-warp blocks measured best)
#endif
constexpr int kRowsWarps = PIC_ROWS_WARPS;
constexpr int kRowsThreads = 32 * kRowsWarps;

template <typename T, int D, int P, int G_>
struct RowsShape {
    static constexpr int S = StencilW<P>::S;
    static constexpr int SZ = (D == 3) ? S : 1;
    static constexpr int ROWS = S * SZ;
    static constexpr int G = ROWS < G_ ? ROWS : G_;              // lanes per item
    static constexpr int RPL = ROWS / G;                         // rows per lane (consecutive, same z)
    static constexpr int NG = 32 / G;                            // items per warp and round
    static constexpr int WR = PIC_ROWS_WR;                       // slots per warp
    static constexpr int kItemMax = 128;                         // particles per item
    static constexpr int REC = (2 * S + SZ + 1 + 3) / 4 * 4;     // elements of a weight record: wx[S] wy[S] wz[SZ] q
    static constexpr int GSTRIDE = G * REC + 16 / sizeof(T);     // +16 bytes: groups start four banks apart
    static constexpr size_t scratch_bytes = sizeof(T) * NG * GSTRIDE;
    static constexpr int kPassCells = 256;                       // cells listed per pass over the range
    static constexpr int kMaxItems = kPassCells + WR / kItemMax + 8;   // every cell one piece + the extra pieces of long runs
    static constexpr size_t item_bytes = sizeof(uint2) * kMaxItems;    // (cell, start | len << 16)
    static constexpr size_t warp_bytes = (scratch_bytes + item_bytes + 16 + 15) / 16 * 16;   // + the item counter
    static constexpr size_t bytes = warp_bytes * kRowsWarps;
    static_assert(RPL >= 1 && RPL <= S, "a lane's rows must share one z plane");
    static_assert(WR <= 65536 && kItemMax < 65536, "start and len of an item are 16-bit fields");
};

// One particle whose cell is not the cell of the run it sits in (cell_offsets that do not describe
// the order): threads-on-particles with global reductions (3.3.4), from registers.
// Out of line and all by value, so that the rare call costs the hot path neither registers nor
// local memory; it stores the advanced particle itself.
template <typename T, int D, int P, int MODE, bool STORE_W>
__device__ __noinline__ void stray_from_regs(T x0, T x1, T x2, T v0, T v1, T v2, T w, int64_t j, GridP<T> g, FieldP<T> f,
                                             PartP<T> dst, double* __restrict__ racc, T dt, T qmdt)
{
    T x[3] = {x0, x1, x2}, v[3] = {v0, v1, v2};
    int first[3] = {0, 0, 0};
    T wt[3][P + 1];
#pragma unroll
    for (int c = 0; c < D; ++c) {
        T t = grid_coord(x[c], g.h[c], g.inv_h[c], g.hmul);
        spline_weights<T, P>(t, cell_index(t, g.n[c]), first[c], wt[c]);
    }
    T e[3] = {(T)0, (T)0, (T)0};
    const T q = (MODE & kModeDeposit) ? w * g.inv_vol : (T)0;
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
            v[c] += qmdt * e[c];
            x[c] = wrap_periodic(x[c] + dt * v[c], g.L[c], g.inv_L[c]);
        }
    }
    if ((MODE & kModePush) || STORE_W) {
#pragma unroll
        for (int c = 0; c < D; ++c) { dst.x[c][j] = x[c]; dst.v[c][j] = v[c]; }
        if (STORE_W) dst.w[j] = w;
    }
}

template <typename T, int D, int P, int MODE, int G_>
constexpr int rows_min_blocks()
{
    return (sizeof(T) == 4 ? PIC_ROWS_MINW32 : 8) / PIC_ROWS_WARPS;
}

template <typename T, int D, int P, int MODE, bool VIA_PERM, int G_>
__global__ void __launch_bounds__(kRowsThreads, (rows_min_blocks<T, D, P, MODE, G_>()))
k_rows(PartP<T> src, PartP<T> dst, const int32_t* __restrict__ perm, GridP<T> g, FieldP<T> f,
       const int32_t* __restrict__ cell_offsets, int64_t n, double* __restrict__ racc, T dt, T qmdt,
       const uint32_t* __restrict__ gate, uint32_t want)
{
    using SH = RowsShape<T, D, P, G_>;
    if (gate && *gate != want) return;                // the caller's cell_offsets failed the device-side check
    constexpr int S = SH::S, S2 = S / 2, SZ = SH::SZ;
    constexpr int G = SH::G, RPL = SH::RPL, NG = SH::NG, WR = SH::WR, REC = SH::REC;
    constexpr int kItemMax = SH::kItemMax;
    constexpr bool DEP = (MODE & kModeDeposit) != 0, PUSH = (MODE & kModePush) != 0;
    constexpr unsigned FULL = 0xFFFFFFFFu;
    constexpr int sh = (S == 4) ? 1 : 0;              // the cell's stencil starts at node i0 - sh

    extern __shared__ __align__(16) unsigned char s_dyn[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int lg = lane % G, grp = lane / G;
    unsigned char* const wsm = s_dyn + (size_t)warp * SH::warp_bytes;
    T* const scratch = reinterpret_cast<T*>(wsm) + grp * SH::GSTRIDE;            // this group's G records
    uint2* const s_item = reinterpret_cast<uint2*>(wsm + SH::scratch_bytes);
    int* const s_nitems = reinterpret_cast<int*>(wsm + SH::scratch_bytes + SH::item_bytes);

    const int64_t j0 = ((int64_t)blockIdx.x * kRowsWarps + warp) * WR;
    if (j0 >= n) return;                              // warps are independent: no block barrier below
    const int cnt = (int)((n - j0 < (int64_t)WR) ? (n - j0) : (int64_t)WR);

    // ---- 1. cells holding the first and the last slot of the range: the key of that particle if
    //         cell_offsets describes the order, else a binary search
    int cfl = 0;
    if (lane < 2) {
        const int64_t j = j0 + (lane == 0 ? 0 : cnt - 1);
        const int64_t i = VIA_PERM ? (int64_t)perm[j] : j;
        int k = 0, mul = 1;
#pragma unroll
        for (int c = 0; c < D; ++c) {
            T t = grid_coord(src.x[c][i], g.h[c], g.inv_h[c], g.hmul);
            k += mul * cell_index(t, g.n[c]);
            mul *= g.n[c];
        }
        if (!((int64_t)cell_offsets[k] <= j && j < (int64_t)cell_offsets[k + 1])) {
            int lo = 0, hi = mul;                     // largest k with cell_offsets[k] <= j
            while (hi - lo > 1) {
                const int mid = lo + (hi - lo) / 2;
                if ((int64_t)cell_offsets[mid] <= j) lo = mid; else hi = mid;
            }
            k = lo;
        }
        cfl = k;
    }
    const int c_first = __shfl_sync(FULL, cfl, 0), c_last = __shfl_sync(FULL, cfl, 1);

    // rows of this lane: r = lg*RPL + rr, z plane kk, y rows jj0 .. jj0+RPL-1
    const int kk = (lg * RPL) / S, jj0 = (lg * RPL) % S;

    // ---- 2. the item list, kPassCells cells at a time: every cell's run inside the range, cut into
    //         pieces of at most kItemMax (a multiple of G except the last piece), in cell order
    for (int cA = c_first; cA <= c_last; cA += SH::kPassCells) {
    const int cB = (c_last - cA < SH::kPassCells) ? c_last : cA + SH::kPassCells - 1;
    __syncwarp();
    if (lane == 0) *s_nitems = 0;
    __syncwarp();
    {
        const int64_t j1 = j0 + cnt;
        for (int cb = cA; cb <= cB; cb += 32) {       // warp-uniform trip count: ballots below
            const int c = cb + lane;
            int len = 0, s = 0;
            if (c <= cB) {
                const int64_t a = cell_offsets[c], b = cell_offsets[c + 1];
                const int64_t lo = a > j0 ? a : j0, hi = b < j1 ? b : j1;
                len = hi > lo ? (int)(hi - lo) : 0;
                s = (int)(lo - j0);
            }
            // pieces of this cell; cells keep their order in the list (neighbouring cells are worked
            // on together: their stencils and particles share cache lines)
            const int nch = (len + kItemMax - 1) / kItemMax;
            int inc = nch;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(FULL, inc, o);
                if (lane >= o) inc += t;
            }
            const int base = *s_nitems;
            const int pos = base + inc - nch;
            if (nch > 0) {
                const int chunk = ((len + nch - 1) / nch + G - 1) / G * G;
                for (int q = 0; q < nch; ++q) {
                    int l = len - q * chunk;
                    l = l < 0 ? 0 : (l < chunk ? l : chunk);
                    s_item[pos + q] = make_uint2((unsigned)c, (unsigned)(s + q * chunk) | ((unsigned)l << 16));
                }
            }
            __syncwarp();
            if (lane == 31) *s_nitems = base + inc;
            __syncwarp();
        }
    }
    const int nitems = *s_nitems;

    // ---- 3. rounds of NG items
    for (int r0 = 0; r0 < nitems; r0 += NG) {
        const int ii = r0 + grp;
        const bool have = ii < nitems;
        const uint2 it = have ? s_item[ii] : make_uint2(0u, 0u);
        const int start = (int)(it.y & 0xFFFFu), len = (int)(it.y >> 16);
        int nbmax = (len + G - 1) / G;
#pragma unroll
        for (int o = 16; o >= G; o >>= 1) nbmax = max(nbmax, __shfl_xor_sync(FULL, nbmax, o));
        if (nbmax == 0) continue;                     // only empty pieces in this round

        // the item's cell and the grid offsets of this lane's nodes
        const int cell = (int)it.x;
        const int cx = cell % g.n[0];
        const int cyz = cell / g.n[0];
        const int cy = (D == 3) ? cyz % g.n[1] : cyz;
        const int cz = (D == 3) ? cyz / g.n[1] : 0;
        int gx[S], rowb[RPL];
#pragma unroll
        for (int i = 0; i < S; ++i) gx[i] = fold(cx - sh + i, g.n[0]);
        {
            const int gz = (D == 3) ? fold(cz - sh + kk, g.n[2]) : 0;
#pragma unroll
            for (int rr = 0; rr < RPL; ++rr) rowb[rr] = g.n[0] * (fold(cy - sh + jj0 + rr, g.n[1]) + g.n[1] * gz);
        }
        // field on this lane's rows, in registers for the whole item
        Pk<T> Er[PUSH ? D : 1][RPL][S2];
        if constexpr (PUSH) {
#pragma unroll
            for (int c = 0; c < D; ++c)
#pragma unroll
                for (int rr = 0; rr < RPL; ++rr)
#pragma unroll
                    for (int i = 0; i < S2; ++i) {
                        const T e0 = have ? __ldg(f.E[c] + rowb[rr] + gx[2 * i]) : (T)0;
                        const T e1 = have ? __ldg(f.E[c] + rowb[rr] + gx[2 * i + 1]) : (T)0;
                        Er[c][rr][i] = pk_make(e0, e1);
                    }
        }
        Pk<T> acc[DEP ? RPL : 1][S2];
#pragma unroll
        for (int rr = 0; rr < (DEP ? RPL : 1); ++rr)
#pragma unroll
            for (int i = 0; i < S2; ++i) acc[rr][i] = pk_zero<T>();

        // particle of this lane in the current batch, and the prefetched one of the next batch
        const int64_t jbase = j0 + start + lg;
        T nx[D], nv[D], nw = (T)0;
#pragma unroll
        for (int c = 0; c < D; ++c) { nx[c] = (T)0; nv[c] = (T)0; }
        int in1 = 0;                                  // source index of this lane's particle in batch b+1 (then b+2)
        auto load_attrs = [&](int i) {
#pragma unroll
            for (int c = 0; c < D; ++c) {
                nx[c] = src.x[c][i];
                if constexpr (PUSH || VIA_PERM) nv[c] = src.v[c][i];
            }
            if constexpr (DEP || VIA_PERM) nw = src.w[i];
        };
        if (have && lg < len) {
            in1 = VIA_PERM ? perm[jbase] : (int)jbase;
            load_attrs(in1);
        }
        if (have && G + lg < len) in1 = VIA_PERM ? perm[jbase + G] : (int)jbase + G;

        for (int b = 0; b < nbmax; ++b) {
            const bool valid = have && b * G + lg < len;
            T px[D], pv[D], pw = nw;
#pragma unroll
            for (int c = 0; c < D; ++c) { px[c] = nx[c]; pv[c] = nv[c]; }
            // prefetch: attributes of batch b+1 (index known), index of batch b+2
            if (have && (b + 1) * G + lg < len) load_attrs(in1);
            // loaded straight into in1 (its old value has just been consumed): no copy of an in-flight load
            if (have && (b + 2) * G + lg < len) in1 = VIA_PERM ? perm[jbase + (b + 2) * G] : (int)jbase + (b + 2) * G;

            // ---- phase W: lane = particle
            bool same = true;
            T q = (T)0;
            {
                T w1[S], w2[S], w3[SZ];
                same = cell_weights<T, P>(px[0], g.h[0], g.inv_h[0], g.hmul, g.n[0], w1) == cx;
                same = (cell_weights<T, P>(px[1], g.h[1], g.inv_h[1], g.hmul, g.n[1], w2) == cy) && same;
                if constexpr (D == 3) {
                    same = (cell_weights<T, P>(px[2], g.h[2], g.inv_h[2], g.hmul, g.n[2], w3) == cz) && same;
                } else {
                    w3[0] = (T)1;
                }
                if constexpr (DEP) q = (valid && same) ? pw * g.inv_vol : (T)0;
                T* const rec = scratch + lg * REC;
                if constexpr (sizeof(T) == 4 && S == 4) {
                    *reinterpret_cast<float4*>(rec) = make_float4(w1[0], w1[1], w1[2], w1[3]);
                    *reinterpret_cast<float4*>(rec + 4) = make_float4(w2[0], w2[1], w2[2], w2[3]);
                    if constexpr (D == 3) {
                        *reinterpret_cast<float4*>(rec + 8) = make_float4(w3[0], w3[1], w3[2], w3[3]);
                        rec[12] = q;
                    } else {
                        rec[8] = w3[0];
                        rec[9] = q;
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < S; ++i) { rec[i] = w1[i]; rec[S + i] = w2[i]; }
#pragma unroll
                    for (int i = 0; i < SZ; ++i) rec[2 * S + i] = w3[i];
                    rec[2 * S + SZ] = q;
                }
            }
            __syncwarp();

            // ---- phase N: lane = rows; all G particles of the batch
            T part[PUSH ? G : 1][D];
#pragma unroll
            for (int p = 0; p < G; ++p) {
                const T* const rp = scratch + p * REC;
                Pk<T> wx2[S2];
                load_row<T, S>(rp, wx2);
                T wyv[RPL];
                if constexpr (RPL == S && S == 4 && sizeof(T) == 4) {
                    const float4 y4 = *reinterpret_cast<const float4*>(rp + S);
                    wyv[0] = y4.x; wyv[1] = y4.y; wyv[2] = y4.z; wyv[3] = y4.w;
                } else {
#pragma unroll
                    for (int rr = 0; rr < RPL; ++rr) wyv[rr] = rp[S + jj0 + rr];
                }
                const T wzv = (D == 3) ? rp[2 * S + kk] : (T)1;
                Pk<T> qv2;
                if constexpr (DEP) { const T qv = rp[2 * S + SZ]; qv2 = pk_make(qv, qv); }
                Pk<T> sum[PUSH ? D : 1];
                bool first = true;
#pragma unroll
                for (int rr = 0; rr < RPL; ++rr) {
                    const T a = wzv * wyv[rr];
                    const Pk<T> a2 = pk_make(a, a);
#pragma unroll
                    for (int i = 0; i < S2; ++i) {
                        const Pk<T> pp = pk_mul(a2, wx2[i]);
                        if constexpr (DEP) acc[rr][i] = pk_fma(qv2, pp, acc[rr][i]);
                        if constexpr (PUSH) {
#pragma unroll
                            for (int c = 0; c < D; ++c) sum[c] = first ? pk_mul(pp, Er[c][rr][i]) : pk_fma(pp, Er[c][rr][i], sum[c]);
                        }
                        first = false;
                    }
                }
                if constexpr (PUSH) {
#pragma unroll
                    for (int c = 0; c < D; ++c) part[p][c] = pk_lo(sum[c]) + pk_hi(sum[c]);
                }
            }
            __syncwarp();

            if constexpr (PUSH) {
                // transposed butterfly: lane lg ends up with the field of particle lg in part[0]
#pragma unroll
                for (int m = G / 2; m >= 1; m >>= 1) {
                    const bool upper = (lg & m) != 0;
#pragma unroll
                    for (int p = 0; p < G / 2; ++p) {
                        if (p < m) {
#pragma unroll
                            for (int c = 0; c < D; ++c) {
                                const T keep = upper ? part[p + m][c] : part[p][c];
                                const T send = upper ? part[p][c] : part[p + m][c];
                                part[p][c] = keep + __shfl_xor_sync(FULL, send, m);
                            }
                        }
                    }
                }
            }

            // ---- accel + push + store (lane = particle again)
            if (valid) {
                const int64_t j = jbase + b * G;
                if (!same) {
                    stray_from_regs<T, D, P, MODE, VIA_PERM>(px[0], px[1], D == 3 ? px[D - 1] : (T)0, pv[0], pv[1],
                                                             D == 3 ? pv[D - 1] : (T)0, pw, j, g, f, dst, racc, dt, qmdt);
                } else if constexpr (PUSH || VIA_PERM) {
                    if constexpr (PUSH) {
                        bool inside = true;
#pragma unroll
                        for (int c = 0; c < D; ++c) {
                            pv[c] += qmdt * part[0][c];
                            px[c] += dt * pv[c];
                            inside = inside && (px[c] >= (T)0 && px[c] < g.L[c]);
                        }
                        if (!inside) {                  // one rare branch for all components
#pragma unroll
                            for (int c = 0; c < D; ++c) px[c] = wrap_periodic(px[c], g.L[c], g.inv_L[c]);
                        }
                    }
#pragma unroll
                    for (int c = 0; c < D; ++c) { dst.x[c][j] = px[c]; dst.v[c][j] = pv[c]; }
                    if constexpr (VIA_PERM) dst.w[j] = pw;
                }
            }
        }

        // ---- end of the item: this lane's node sums go to the grid
        if constexpr (DEP) {
            if (have) {
#pragma unroll
                for (int rr = 0; rr < RPL; ++rr)
#pragma unroll
                    for (int i = 0; i < S2; ++i) {
                        atomicAdd(&racc[rowb[rr] + gx[2 * i]], (double)pk_lo(acc[rr][i]));
                        atomicAdd(&racc[rowb[rr] + gx[2 * i + 1]], (double)pk_hi(acc[rr][i]));
                    }
            }
        }
    }
    }   // passes over the cells of the range
}

// launch k_rows over n particles sorted by cell.  VIA_PERM: particle perm[j] of src -> slot j of dst;
// otherwise in place on dst.  racc = double accumulation grid of the deposit.
template <typename T, int D, int P, int MODE, bool VIA_PERM>
inline int launch_rows(const pic_grid_t& g, const pic_particles_t& src, const pic_particles_t& dst,
                       const int32_t* perm, const int32_t* cell_offsets, const void* const E[3], double* racc,
                       double dt, double qm, cudaStream_t st, const uint32_t* gate = nullptr, uint32_t want = 0)
{
    if (dst.n <= 0) return PIC_OK;
    constexpr int GP = sizeof(T) == 4 ? PIC_ROWS_G32 : 8;
    using SH = RowsShape<T, D, P, GP>;
    FieldP<T> f;
    for (int c = 0; c < 3; ++c) f.E[c] = (E && c < D) ? (const T*)E[c] : nullptr;
    auto kern = k_rows<T, D, P, MODE, VIA_PERM, GP>;
    constexpr size_t smem = SH::bytes;
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return PIC_ERR_CUDA;
        attr_set = true;
    }
    constexpr int64_t per_block = (int64_t)SH::WR * kRowsWarps;
    const unsigned blocks = (unsigned)((dst.n + per_block - 1) / per_block);
    kern<<<blocks, kRowsThreads, smem, st>>>(make_partp<T>(VIA_PERM ? src : dst), make_partp<T>(dst), perm,
                                            make_gridp<T>(g), f, cell_offsets, dst.n, racc, (T)dt, (T)(qm * dt), gate, want);
    count_launch();
    return cudaGetLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

}  // namespace pic
