// pic_tile.cuh -- the step pass for particles sorted into BUCKETS OF SEVERAL CELLS (pic_step_buckets, NEXT-2): a block
// stages its bucket's grid tile in shared memory, the paper's own CUDA design.
//
// "An optimization of this algorithm is possible in CUDA by using shared memory as an intermediate step to do the
// reduction ... sorting is required and the reduction is done with two steps: first with CUDA to shared memory, then
// from shared memory to global memory where the grid is stored" (section 3.3.4; kernel of App. B,
// `rholoc` tile with guard nodes, atomicAdd into it, flush with atomicAdd to `rho`).  The field is
// staged the same way for the gather (north_star: "smem-staged field stencils").
//
//   * block (b, r): bucket b, share r of its particles (R blocks per bucket, R from the mean bucket population, so that
//     few large buckets still fill the machine).  The bucket covers cells [o_c, o_c + e_c) per dimension; its particles
//     touch the nodes o_c - lo .. o_c + e_c - 1 + hi (lo, hi = 0, 1 for p = 1; 1, 2 for p = 2, 3): the tile.
//   * stage: E[c] on the tile's nodes (folded periodically) -> shared memory; rho tile = 0.
//   * threads on particles (setrho 3.3.4): weights, (p+1)^d atomic adds into the shared rho tile -- in DOUBLE, like every
//     deposit of this library, so that the result does not depend on the density -- and (p+1)^d reads of the shared field
//     per component; accel, push, wrap, store.  Inside a bucket the order of the particles does not matter.
//   * flush: every tile node with a non-zero sum goes to the global double grid with one atomic add.
//
// Shared-memory floating-point atomics are compare-and-swap loops on sm_100a, and neighbouring particles of a warp read
// different tile nodes (bank conflicts): this kernel is the measured counterpart of k_runs (one cell per bucket, no
// shared-memory atomics), see profiles/ and DESIGN.md.  Buckets whose tile does not fit in shared memory fall back to
// k_runs<STRAYS>.
#pragma once
#include "pic_stencil.cuh"

namespace pic {

constexpr int kTileThreads = 256;
constexpr size_t kTileMaxBytes = 160 * 1024;

// nodes of the largest tile of this bucket shape, and its shared-memory bytes (E: d values of T, rho: one double)
template <typename T>
inline size_t tile_bytes(const pic_grid_t& g, const int32_t* bucket)
{
    size_t nodes = 1;
    for (int c = 0; c < g.dim; ++c) nodes *= (size_t)(bucket[c] + (g.order == 1 ? 1 : 3));
    return nodes * (sizeof(double) + (size_t)g.dim * sizeof(T)) + 16;
}

template <typename T, int D, int P, bool VIA_PERM>
__global__ void __launch_bounds__(kTileThreads)
k_bucket_tile(PartP<T> src, PartP<T> dst, const int32_t* __restrict__ perm, const int32_t* __restrict__ bucket_off, GridP<T> g,
              FieldP<T> f, double* __restrict__ racc, double dtd, double qmdtd, int R, const uint32_t* __restrict__ gate, uint32_t want)
{
    if (gate && *gate != want) return;
    extern __shared__ __align__(16) unsigned char s_tile[];
    constexpr int lo = (P == 1) ? 0 : 1, ext = (P == 1) ? 1 : 3;      // tile = cells' nodes - lo .. + ext - lo
    const T dt = (T)dtd, qmdt = (T)qmdtd;
    const int b = blockIdx.x / R, r = blockIdx.x - b * R;
    int o[3] = {0, 0, 0}, t[3] = {1, 1, 1};                           // first cell of the bucket, tile nodes per dimension
    {
        int q = b;
#pragma unroll
        for (int c = 0; c < D; ++c) {
            const int bc = q % g.nbk[c];
            q /= g.nbk[c];
            o[c] = bc * g.bk[c];
            const int e = min(g.bk[c], g.n[c] - o[c]);
            t[c] = e + ext;
        }
    }
    const int nodes = t[0] * t[1] * t[2];
    double* s_rho = reinterpret_cast<double*>(s_tile);                // [nodes]
    T* s_E = reinterpret_cast<T*>(s_rho + nodes);                     // [D][nodes]
    const int32_t p0 = bucket_off[b], p1 = bucket_off[b + 1];
    const int32_t cnt = p1 - p0, chunk = (cnt + R - 1) / R;
    const int32_t j0 = p0 + r * chunk, j1 = min(p1, j0 + chunk);
    if (j0 >= j1) return;                                             // (whole block: no barrier is skipped by a part of it)

    for (int k = threadIdx.x; k < nodes; k += kTileThreads) {
        const int lx = k % t[0], ly = (k / t[0]) % t[1], lz = k / (t[0] * t[1]);
        const int gx = fold(o[0] - lo + lx, g.n[0]) , gy = fold(o[1] - lo + ly, g.n[1]);
        const int gz = (D == 3) ? fold(o[2] - lo + lz, g.n[2]) : 0;
        const int64_t at = gx + (int64_t)g.n[0] * (gy + (int64_t)g.n[1] * gz);
        s_rho[k] = 0.0;
#pragma unroll
        for (int c = 0; c < D; ++c) s_E[c * nodes + k] = __ldg(f.E[c] + at);
    }
    __syncthreads();

    for (int32_t j = j0 + threadIdx.x; j < j1; j += kTileThreads) {
        const int64_t i = VIA_PERM ? (int64_t)perm[j] : (int64_t)j;
        T x[D], v[D], e[D];
        int li[3] = {0, 0, 0};
        T wt[3][P + 1];
#pragma unroll
        for (int c = 0; c < D; ++c) {
            x[c] = src.x[c][i];
            v[c] = src.v[c][i];
            e[c] = (T)0;
            const T tt = grid_coord(x[c], g.h[c], g.inv_h[c], g.hmul);
            int first;
            spline_weights<T, P>(tt, cell_index(tt, g.n[c]), first, wt[c]);
            li[c] = first - (o[c] - lo);                              // local node of the first stencil point: 0 .. t - P - 1
        }
        const T w = src.w[i];
        const T q = w * g.inv_vol;
        constexpr int PZ = (D == 3) ? P : 0;
#pragma unroll
        for (int cz = 0; cz <= PZ; ++cz) {
            const T wz = (D == 3) ? wt[2][cz] : (T)1;
#pragma unroll
            for (int cy = 0; cy <= P; ++cy) {
                const T wyz = wz * wt[1][cy];
                const int row = t[0] * ((li[1] + cy) + t[1] * (li[2] + cz)) + li[0];
#pragma unroll
                for (int cx = 0; cx <= P; ++cx) {
                    const T wgt = wyz * wt[0][cx];
                    atomicAdd(&s_rho[row + cx], (double)(q * wgt));
#pragma unroll
                    for (int c = 0; c < D; ++c) e[c] += wgt * s_E[c * nodes + row + cx];
                }
            }
        }
#pragma unroll
        for (int c = 0; c < D; ++c) {
            const T vn = v[c] + qmdt * e[c];
            T xn = x[c] + dt * vn;
            if (!(xn >= (T)0 && xn < g.L[c])) xn = advance_wrap<T>(x[c], v[c], e[c], dtd, qmdtd, g.Ld[c]);
            dst.x[c][j] = xn;
            dst.v[c][j] = vn;
        }
        if constexpr (VIA_PERM) dst.w[j] = w;
    }
    __syncthreads();

    for (int k = threadIdx.x; k < nodes; k += kTileThreads) {
        const double s = s_rho[k];
        if (s != 0.0) {
            const int lx = k % t[0], ly = (k / t[0]) % t[1], lz = k / (t[0] * t[1]);
            const int gx = fold(o[0] - lo + lx, g.n[0]), gy = fold(o[1] - lo + ly, g.n[1]);
            const int gz = (D == 3) ? fold(o[2] - lo + lz, g.n[2]) : 0;
            atomicAdd(&racc[gx + (int64_t)g.n[0] * (gy + (int64_t)g.n[1] * gz)], s);
        }
    }
}

// One pass over particles in bucket order.  VIA_PERM: particle perm[j] of src -> slot j of dst, else in place on dst.
// Returns PIC_ERR_UNSUPPORTED if the tile does not fit (the caller then takes the run kernel).
template <typename T, int D, int P, bool VIA_PERM>
inline int launch_bucket_tile(const pic_grid_t& g, const int32_t* bucket, int64_t nbuckets, const pic_particles_t& src,
                              const pic_particles_t& dst, const int32_t* perm, const int32_t* bucket_off, const void* const E[3],
                              double* racc, double dt, double qm, cudaStream_t st, const uint32_t* gate, uint32_t want)
{
    if (dst.n <= 0) return PIC_OK;
    const size_t smem = tile_bytes<T>(g, bucket);
    if (smem > kTileMaxBytes) return PIC_ERR_UNSUPPORTED;
    int64_t R = (dst.n / nbuckets + 4095) / 4096;                  // blocks per bucket: about 4096 particles each ...
    const int64_t fill = ((int64_t)sm_count() * 4 + nbuckets - 1) / nbuckets;   // ... and at least four blocks per SM
    if (R < fill) R = fill;
    if (R < 1) R = 1;
    if (R > 1024) R = 1024;
    if (nbuckets * R >= ((int64_t)1 << 31)) return PIC_ERR_UNSUPPORTED;
    FieldP<T> f;
    for (int c = 0; c < 3; ++c) f.E[c] = (E && c < D) ? (const T*)E[c] : nullptr;
    auto kern = k_bucket_tile<T, D, P, VIA_PERM>;
    if (smem > 48 * 1024) PIC_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<(unsigned)(nbuckets * R), kTileThreads, smem, st>>>(make_partp<T>(VIA_PERM ? src : dst), make_partp<T>(dst), perm, bucket_off,
                                                               make_gridp<T>(g, bucket), f, racc, dt, qm * dt, (int)R, gate, want);
    count_launch();
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

}  // namespace pic
