// pic_group.cuh -- the sorted-order kernel: deposit and/or gather+accel+push over particles that
// are grouped by cell (rows a5-a7, their fusion a8, optionally fused with the reorder a4).
//
// Prior art: the paper's CUDA kernel stages a per-block tile of rho in shared memory and
// atomicAdds every particle's 8 products into it ("sorting is required"),
// and notes the alternative of reducing "on a temporary thread-private variable without atomics",
// putting the result "only once with atomic adds to the grid".  On sm_100a a
// floating-point atomicAdd on shared memory is a compare-and-swap loop, so this kernel takes the
// second road: LANE = PARTICLE, a GROUP of G = 8 lanes = one cell.
//
//   * a warp owns WR consecutive slots of the sorted order and lists the cell runs inside them
//     ("items", at most kItemMax particles).  No block-level barrier anywhere: warps are independent.
//   * the four groups of a warp take four items at a time.  A group first stages the field stencil
//     of its cell (S^d nodes x d components, read-only loads) in its shared-memory
//     slot, then walks through the item G particles at a time.  Every lane reads its particle
//     straight from global memory (through perm when the reorder is fused in; the next batch is
//     prefetched into registers), computes the 1-D spline weights, and in one loop over the
//     S^(d-1) stencil rows adds w*W to its PRIVATE node sums (registers) and W*E to its gather sums,
//     the field rows coming from shared memory by broadcast 128-bit loads.  Then accel, push, store.
//   * at the end of the item the G lanes write their S^d node sums to the group's slot, every lane
//     adds up the G copies of the nodes it owns and sends the totals to the grid with global
//     reductions (RED) in double precision, so that the result does not depend on the density.
//
// S = stencil width of a CELL: 2 for p = 1, 4 for p = 2, 3 (a quadratic particle touches 3 of the
// 4 nodes i0-1..i0+2, which 3 depends on xi >= 1/2; the fourth weight is an exact zero).
// Arithmetic on pairs of x-neighbouring nodes uses the packed fp32 instructions of sm_100
// (fma.rn.f32x2): same FMA-pipe time, half the issue slots.
#pragma once
#include "pic_rows.cuh"

namespace pic {

#ifndef PIC_GRP_MINB32
#define PIC_GRP_MINB32 3        // resident blocks per SM the fp32 kernels are compiled for
#endif
#ifndef PIC_GRP_WR
#define PIC_GRP_WR 2048         // slots of the sorted order per warp
#endif
constexpr int kGrpWarps = 4;
constexpr int kGrpThreads = 32 * kGrpWarps;

__device__ __forceinline__ Pk<float> pk_add(Pk<float> a, Pk<float> b)
{
    Pk<float> d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d.r) : "l"(a.r), "l"(b.r));
    return d;
}
__device__ __forceinline__ Pk<double> pk_add(Pk<double> a, Pk<double> b) { return Pk<double>{a.lo + b.lo, a.hi + b.hi}; }

// S consecutive values to shared memory from S/2 pairs (128-bit stores where possible)
template <typename T, int S>
__device__ __forceinline__ void store_row(T* __restrict__ p, const Pk<T> (&e)[S / 2])
{
    if constexpr (sizeof(T) == 4 && S == 4) {
        *reinterpret_cast<float4*>(p) = make_float4(pk_lo(e[0]), pk_hi(e[0]), pk_lo(e[1]), pk_hi(e[1]));
    } else if constexpr (sizeof(T) == 4) {
        *reinterpret_cast<float2*>(p) = make_float2(pk_lo(e[0]), pk_hi(e[0]));
    } else {
#pragma unroll
        for (int i = 0; i < S / 2; ++i) *reinterpret_cast<double2*>(p + 2 * i) = make_double2(pk_lo(e[i]), pk_hi(e[i]));
    }
}

// asynchronous 4- or 8-byte copy global -> shared (LDGSTS): no register staging
template <typename T>
__device__ __forceinline__ void cp_async_elem(T* smem_dst, const T* gmem_src)
{
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    if constexpr (sizeof(T) == 4)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(sa), "l"(gmem_src) : "memory");
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

template <typename T, int D, int P>
struct GroupShape {
    static constexpr int S = StencilW<P>::S;
    static constexpr int S2 = S / 2;
    static constexpr int SZ = (D == 3) ? S : 1;
    static constexpr int ROWS = S * SZ;
    static constexpr int NODES = ROWS * S;
    static constexpr int G = 8;                                   // lanes per item
    static constexpr int NG = 32 / G;                             // items per warp and round
    static constexpr int VEC = 16 / sizeof(T);                    // elements per 128-bit access
    static constexpr int CW = S < VEC ? S : VEC;                  // a chunk: CW x-neighbouring nodes of one row
    static constexpr int NCH = NODES / CW;                        // chunks of a stencil
    static constexpr int CPL = (NCH + G - 1) / G;                 // chunks a lane owns: lg, lg+G, ...
    static constexpr int CSTRIDE = NODES + VEC;                   // one lane's node sums (+16 B: lanes four banks apart)
    static constexpr int EBUF = D * NODES;                        // one field stencil; two buffers (this round, next round)
    static constexpr int slot_elems()
    {
        int e = 2 * EBUF + G * CSTRIDE;                           // field stencils | node sums of the G lanes
        while ((e * (int)sizeof(T)) % 128 != 16) e += VEC;        // groups start four banks apart
        return e;
    }
    static constexpr int GSLOT = slot_elems();
    static constexpr int WR = PIC_GRP_WR;                         // slots per warp
    static constexpr int kItemMax = 128;                          // particles per item
    static constexpr int kPassCells = 128;                        // cells listed per pass over the range
    static constexpr int kMaxItems = kPassCells + WR / kItemMax + 8;
    static constexpr size_t scratch_bytes = sizeof(T) * NG * GSLOT;
    static constexpr size_t item_bytes = sizeof(uint2) * kMaxItems;   // (cell, start | len << 16)
    static constexpr size_t warp_bytes = (scratch_bytes + item_bytes + 16 + 15) / 16 * 16;
    static constexpr size_t bytes = warp_bytes * kGrpWarps;
    static constexpr int min_blocks = sizeof(T) == 4 ? PIC_GRP_MINB32 : 2;   // resident blocks per SM the kernel is compiled for
    static_assert(WR <= 65536 && kItemMax < 65536, "start and len of an item are 16-bit fields");
    static_assert(NODES % CW == 0 && S % CW == 0, "a chunk lies inside one stencil row");
};

template <typename T, int D, int P, int MODE, bool VIA_PERM>
__global__ void __launch_bounds__(kGrpThreads, (GroupShape<T, D, P>::min_blocks))
k_group(PartP<T> src, PartP<T> dst, const int32_t* __restrict__ perm, GridP<T> g, FieldP<T> f,
        const int32_t* __restrict__ cell_offsets, int64_t n, double* __restrict__ racc, T dt, T qmdt)
{
    using SH = GroupShape<T, D, P>;
    constexpr int S = SH::S, S2 = SH::S2, SZ = SH::SZ, ROWS = SH::ROWS, NODES = SH::NODES;
    constexpr int G = SH::G, NG = SH::NG, WR = SH::WR, CW = SH::CW, NCH = SH::NCH, CPL = SH::CPL;
    constexpr int kItemMax = SH::kItemMax;
    constexpr bool DEP = (MODE & kModeDeposit) != 0, PUSH = (MODE & kModePush) != 0;
    constexpr unsigned FULL = 0xFFFFFFFFu;
    constexpr int sh = (S == 4) ? 1 : 0;              // the cell's stencil starts at node i0 - sh

    extern __shared__ __align__(16) unsigned char s_dyn[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int lg = lane % G, grp = lane / G;
    unsigned char* const wsm = s_dyn + (size_t)warp * SH::warp_bytes;
    T* const slot = reinterpret_cast<T*>(wsm) + grp * SH::GSLOT;                 // this group's field buffers
    T* const sums = slot + 2 * SH::EBUF;                                         // this group's node sums
    uint2* const s_item = reinterpret_cast<uint2*>(wsm + SH::scratch_bytes);
    int* const s_nitems = reinterpret_cast<int*>(wsm + SH::scratch_bytes + SH::item_bytes);

    const int64_t j0 = ((int64_t)blockIdx.x * kGrpWarps + warp) * WR;
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

    // grid offsets of the nodes this lane owns in the stencil of `cell` (chunks lg, lg+G, ...)
    auto chunk_offsets = [&](int cell, int (&coff)[CPL][CW]) {
        const int cx = cell % g.n[0];
        const int cyz = cell / g.n[0];
        const int cy = (D == 3) ? cyz % g.n[1] : cyz;
        const int cz = (D == 3) ? cyz / g.n[1] : 0;
#pragma unroll
        for (int q = 0; q < CPL; ++q) {
            const int ch = q * G + lg;
            const int row = (ch * CW) / S, i0 = (ch * CW) % S;
            const int jj = row % S, kk = row / S;
            const int gz = (D == 3) ? fold(cz - sh + kk, g.n[2]) : 0;
            const int rowb = g.n[0] * (fold(cy - sh + jj, g.n[1]) + g.n[1] * gz);
#pragma unroll
            for (int e = 0; e < CW; ++e) coff[q][e] = rowb + fold(cx - sh + i0 + e, g.n[0]);
        }
    };
    // the field stencil of `cell`, first into registers (read-only loads) ...
    auto stage_load = [&](int cell, T (&ev)[CPL][PUSH ? D : 1][CW]) {
        int coff[CPL][CW];
        chunk_offsets(cell, coff);
#pragma unroll
        for (int q = 0; q < CPL; ++q) {
            const int ch = q * G + lg;
            if (NCH % G == 0 || ch < NCH) {
#pragma unroll
                for (int c = 0; c < (PUSH ? D : 1); ++c)
#pragma unroll
                    for (int e = 0; e < CW; ++e) ev[q][c][e] = __ldg(f.E[c] + coff[q][e]);
            }
        }
    };
    // ... then into a field buffer: buf[c*NODES + node]
    auto stage_store = [&](const T (&ev)[CPL][PUSH ? D : 1][CW], T* buf) {
#pragma unroll
        for (int q = 0; q < CPL; ++q) {
            const int ch = q * G + lg;
            if (NCH % G == 0 || ch < NCH) {
#pragma unroll
                for (int c = 0; c < (PUSH ? D : 1); ++c) {
                    Pk<T> pr[CW / 2];
#pragma unroll
                    for (int e = 0; e < CW / 2; ++e) pr[e] = pk_make(ev[q][c][2 * e], ev[q][c][2 * e + 1]);
                    store_row<T, CW>(buf + c * NODES + ch * CW, pr);
                }
            }
        }
    };

    // ---- 2. the item list, kPassCells cells at a time: every cell's run inside the range, cut into
    //         pieces of at most kItemMax (a multiple of G except the last piece), in cell order
    for (int cA = c_first; cA <= c_last; cA += SH::kPassCells) {
    const int cB = (c_last - cA < SH::kPassCells) ? c_last : cA + SH::kPassCells - 1;
    __syncwarp();
    if (lane == 0) *s_nitems = 0;
    __syncwarp();
    {
        const int64_t j1 = j0 + cnt;
        for (int cb = cA; cb <= cB; cb += 32) {       // warp-uniform trip count
            const int c = cb + lane;
            int len = 0, s = 0;
            if (c <= cB) {
                const int64_t a = cell_offsets[c], b = cell_offsets[c + 1];
                const int64_t lo = a > j0 ? a : j0, hi = b < j1 ? b : j1;
                len = hi > lo ? (int)(hi - lo) : 0;
                s = (int)(lo - j0);
            }
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
                    if (l > 0) s_item[pos + q] = make_uint2((unsigned)c, (unsigned)(s + q * chunk) | ((unsigned)l << 16));
                    else s_item[pos + q] = make_uint2((unsigned)c, (unsigned)s);
                }
            }
            __syncwarp();
            if (lane == 31) *s_nitems = base + inc;
            __syncwarp();
        }
    }
    const int nitems = *s_nitems;

    // ---- 3. rounds of NG items.  The lane's particles form one stream across the rounds: the
    //         attributes of its next particle and the perm entry of the one after are in flight
    //         while the current one is worked on; each carries the slot it belongs to (a tag), so
    //         a particle that was not prefetched is simply loaded when it is needed.
    T nx[D], nv[D], nw = (T)0;
#pragma unroll
    for (int c = 0; c < D; ++c) { nx[c] = (T)0; nv[c] = (T)0; }
    int tag_attr = -1, tag_perm = -1, pre_perm = 0;  // slots (relative to j0) of the prefetched attributes / perm entry
    auto load_attrs = [&](int64_t i) {
#pragma unroll
        for (int c = 0; c < D; ++c) {
            nx[c] = src.x[c][i];
            if constexpr (PUSH || VIA_PERM) nv[c] = src.v[c][i];
        }
        if constexpr (DEP || VIA_PERM) nw = src.w[i];
    };
    auto source_of = [&](int rel) -> int64_t {      // source index of the particle in slot j0 + rel
        if constexpr (VIA_PERM) return (rel == tag_perm) ? (int64_t)pre_perm : (int64_t)perm[j0 + rel];
        else return j0 + rel;
    };
    if constexpr (PUSH) {
        if (grp < nitems) {
            T ev[CPL][D][CW];
            stage_load((int)s_item[grp].x, ev);
            stage_store(ev, slot);
        }
    }
    int ebuf = 0;
    for (int r0 = 0; r0 < nitems; r0 += NG, ebuf ^= 1) {
        const int ii = r0 + grp;
        const bool have = ii < nitems;
        const uint2 it = have ? s_item[ii] : make_uint2(0u, 0u);
        const int start = (int)(it.y & 0xFFFFu), len = (int)(it.y >> 16);
        const bool have_n = ii + NG < nitems;
        const uint2 itn = have_n ? s_item[ii + NG] : make_uint2(0u, 0u);
        const int start_n = (int)(itn.y & 0xFFFFu), len_n = (int)(itn.y >> 16);
        const int nb_lane = len > lg ? (len - lg + G - 1) / G : 0;          // batches in which this lane has a particle
        const int nb_lane_n = len_n > lg ? (len_n - lg + G - 1) / G : 0;
        int nbmax = (len + G - 1) / G;
#pragma unroll
        for (int o = 16; o >= G; o >>= 1) nbmax = max(nbmax, __shfl_xor_sync(FULL, nbmax, o));
        // slot (relative to j0) of the lane's k-th particle after batch b, -1 if there is none in sight
        auto slot_ahead = [&](int bb) -> int {
            if (bb < nb_lane) return start + bb * G + lg;
            bb -= nb_lane;
            return bb < nb_lane_n ? start_n + bb * G + lg : -1;
        };

        const int cell = (int)it.x;
        const int cx = cell % g.n[0];
        const int cyz = cell / g.n[0];
        const int cy = (D == 3) ? cyz % g.n[1] : cyz;
        const int cz = (D == 3) ? cyz / g.n[1] : 0;
        T* const fE = slot + ebuf * SH::EBUF;        // this round's field stencil
        if constexpr (PUSH) {
            __syncwarp();                               // the stencil staged at the end of the previous round
        }

        Pk<T> acc[DEP ? NODES / 2 : 1];
#pragma unroll
        for (int a = 0; a < (DEP ? NODES / 2 : 1); ++a) acc[a] = pk_zero<T>();

        for (int b = 0; b < nbmax; ++b) {
            const bool valid = b < nb_lane;
            const int rel = start + b * G + lg;
            T px[D], pv[D], pw;
            if (valid) {
                if (tag_attr != rel) load_attrs(source_of(rel));
#pragma unroll
                for (int c = 0; c < D; ++c) { px[c] = nx[c]; pv[c] = nv[c]; }
                pw = nw;
                // prefetch: attributes of the lane's next particle, perm entry of the one after
                const int r1 = slot_ahead(b + 1), r2 = slot_ahead(b + 2);
                if (r1 >= 0) { load_attrs(source_of(r1)); tag_attr = r1; }
                if constexpr (VIA_PERM) {
                    if (r2 >= 0) { pre_perm = perm[j0 + r2]; tag_perm = r2; }
                }
            } else {
#pragma unroll
                for (int c = 0; c < D; ++c) { px[c] = (T)0; pv[c] = (T)0; }
                pw = (T)0;
            }

            T w1[S], w2[S], w3[SZ];
            bool same = cell_weights<T, P>(px[0], g.h[0], g.inv_h[0], g.hmul, g.n[0], w1) == cx;
            same = (cell_weights<T, P>(px[1], g.h[1], g.inv_h[1], g.hmul, g.n[1], w2) == cy) && same;
            if constexpr (D == 3) {
                same = (cell_weights<T, P>(px[2], g.h[2], g.inv_h[2], g.hmul, g.n[2], w3) == cz) && same;
            } else {
                w3[0] = (T)1;
            }
            Pk<T> wx2[S2], qwx2[DEP ? S2 : 1];
#pragma unroll
            for (int i = 0; i < S2; ++i) wx2[i] = pk_make(w1[2 * i], w1[2 * i + 1]);
            if constexpr (DEP) {
                const T q = (valid && same) ? pw * g.inv_vol : (T)0;
                const Pk<T> q2 = pk_make(q, q);
#pragma unroll
                for (int i = 0; i < S2; ++i) qwx2[i] = pk_mul(q2, wx2[i]);
            }
            Pk<T> sg[PUSH ? D : 1][S2];              // gather sums per x-node pair
            if constexpr (PUSH) {
#pragma unroll
                for (int c = 0; c < D; ++c)
#pragma unroll
                    for (int i = 0; i < S2; ++i) sg[c][i] = pk_zero<T>();
            }
            // field rows are read one row ahead of their use
            Pk<T> er[2][PUSH ? D : 1][S2];
            if constexpr (PUSH) {
#pragma unroll
                for (int c = 0; c < D; ++c) load_row<T, S>(fE + c * NODES, er[0][c]);
            }
#pragma unroll
            for (int row = 0; row < ROWS; ++row) {
                const int kk = row / S, jj = row % S;
                if constexpr (PUSH) {
                    if (row + 1 < ROWS) {
#pragma unroll
                        for (int c = 0; c < D; ++c) load_row<T, S>(fE + c * NODES + (row + 1) * S, er[(row + 1) & 1][c]);
                    }
                }
                const T wyz = w3[kk] * w2[jj];
                const Pk<T> wyz2 = pk_make(wyz, wyz);
                if constexpr (DEP) {
#pragma unroll
                    for (int i = 0; i < S2; ++i) acc[row * S2 + i] = pk_fma(wyz2, qwx2[i], acc[row * S2 + i]);
                }
                if constexpr (PUSH) {
#pragma unroll
                    for (int c = 0; c < D; ++c)
#pragma unroll
                        for (int i = 0; i < S2; ++i) sg[c][i] = pk_fma(wyz2, er[row & 1][c][i], sg[c][i]);
                }
            }

            // ---- accel + push + store
            if (valid) {
                const int64_t j = j0 + rel;
                if (!same) {
                    stray_from_regs<T, D, P, MODE, VIA_PERM>(px[0], px[1], D == 3 ? px[D - 1] : (T)0, pv[0], pv[1],
                                                             D == 3 ? pv[D - 1] : (T)0, pw, j, g, f, dst, racc, dt, qmdt);
                } else if constexpr (PUSH || VIA_PERM) {
                    if constexpr (PUSH) {
                        bool inside = true;
#pragma unroll
                        for (int c = 0; c < D; ++c) {
                            Pk<T> t2 = pk_mul(sg[c][0], wx2[0]);
#pragma unroll
                            for (int i = 1; i < S2; ++i) t2 = pk_fma(sg[c][i], wx2[i], t2);
                            pv[c] += qmdt * (pk_lo(t2) + pk_hi(t2));
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

        // the next round's field stencil is fetched while the node sums are combined
        T evn[CPL][PUSH ? D : 1][CW];
        if constexpr (PUSH) {
            if (have_n) stage_load((int)itn.x, evn);
        }

        // ---- end of the item: the G lanes' node sums meet in shared memory; every lane adds up the
        //      G copies of the chunks it owns and sends the totals to the grid
        if constexpr (DEP) {
            T* const mine = sums + lg * SH::CSTRIDE;
#pragma unroll
            for (int row = 0; row < ROWS; ++row) {
                Pk<T> rv[S2];
#pragma unroll
                for (int i = 0; i < S2; ++i) rv[i] = acc[row * S2 + i];
                store_row<T, S>(mine + row * S, rv);
            }
            __syncwarp();
            int coff[CPL][CW];
            chunk_offsets(cell, coff);
#pragma unroll
            for (int q = 0; q < CPL; ++q) {
                const int ch = q * G + lg;
                if (have && (NCH % G == 0 || ch < NCH)) {
                    Pk<T> tot[CW / 2];
                    load_row<T, CW>(sums + ch * CW, tot);
#pragma unroll
                    for (int l = 1; l < G; ++l) {
                        Pk<T> t[CW / 2];
                        load_row<T, CW>(sums + l * SH::CSTRIDE + ch * CW, t);
#pragma unroll
                        for (int e = 0; e < CW / 2; ++e) tot[e] = pk_add(tot[e], t[e]);
                    }
#pragma unroll
                    for (int e = 0; e < CW / 2; ++e) {
                        atomicAdd(&racc[coff[q][2 * e]], (double)pk_lo(tot[e]));
                        atomicAdd(&racc[coff[q][2 * e + 1]], (double)pk_hi(tot[e]));
                    }
                }
            }
            __syncwarp();                               // before the next item's sums are written
        }
        if constexpr (PUSH) {
            if (have_n) stage_store(evn, slot + (ebuf ^ 1) * SH::EBUF);
        }
    }
    __syncwarp();
    }   // passes over the cells of the range
}

// launch k_group over n particles sorted by cell.  VIA_PERM: particle perm[j] of src -> slot j of dst;
// otherwise in place on dst.  racc = double accumulation grid of the deposit.
template <typename T, int D, int P, int MODE, bool VIA_PERM>
inline int launch_group(const pic_grid_t& g, const pic_particles_t& src, const pic_particles_t& dst,
                        const int32_t* perm, const int32_t* cell_offsets, const void* const E[3], double* racc,
                        double dt, double qm, cudaStream_t st)
{
    if (dst.n <= 0) return PIC_OK;
    using SH = GroupShape<T, D, P>;
    FieldP<T> f;
    for (int c = 0; c < 3; ++c) f.E[c] = (E && c < D) ? (const T*)E[c] : nullptr;
    auto kern = k_group<T, D, P, MODE, VIA_PERM>;
    constexpr size_t smem = SH::bytes;
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return PIC_ERR_CUDA;
        attr_set = true;
    }
    constexpr int64_t per_block = (int64_t)SH::WR * kGrpWarps;
    const unsigned blocks = (unsigned)((dst.n + per_block - 1) / per_block);
    kern<<<blocks, kGrpThreads, smem, st>>>(make_partp<T>(VIA_PERM ? src : dst), make_partp<T>(dst), perm,
                                           make_gridp<T>(g), f, cell_offsets, dst.n, racc, (T)dt, (T)(qm * dt));
    count_launch();
    return cudaGetLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

// the sorted-order kernel the entry points use (PIC_SORTED_KERNEL = 0: k_group, 1: k_rows)
#ifndef PIC_SORTED_KERNEL
#define PIC_SORTED_KERNEL 1
#endif
template <typename T, int D, int P, int MODE, bool VIA_PERM>
inline int launch_sorted(const pic_grid_t& g, const pic_particles_t& src, const pic_particles_t& dst,
                         const int32_t* perm, const int32_t* cell_offsets, const void* const E[3], double* racc,
                         double dt, double qm, cudaStream_t st, const uint32_t* gate = nullptr, uint32_t want = 0)
{
#if PIC_SORTED_KERNEL == 1
    return launch_rows<T, D, P, MODE, VIA_PERM>(g, src, dst, perm, cell_offsets, E, racc, dt, qm, st, gate, want);
#else
    return launch_group<T, D, P, MODE, VIA_PERM>(g, src, dst, perm, cell_offsets, E, racc, dt, qm, st);
#endif
}

}  // namespace pic
