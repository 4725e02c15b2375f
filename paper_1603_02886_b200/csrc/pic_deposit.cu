// pic_deposit.cu -- charge deposition, setrho (row a5).
//
//   rho[j] = h^-d sum_i w_i prod_c W_p(x_ic/h_c - j_c)      (PAPER.md:79 step i; R2 for w and h^-d)
//
// k_deposit_particles is the paper's collision-resolving "threads on particles" algorithm
// (setrho 3.3.4): one thread per particle, (p+1)^d atomic adds to the grid.
// It is correct for ANY particle order and is the path for PIC_ORDER_UNSORTED input.
// Particles in cell order (PIC_ORDER_SORTED / STALE) go through k_runs (pic_runs.cuh).
#include "pic_runs.cuh"

namespace pic {

template <typename T, int D, int P>
__global__ void __launch_bounds__(256) k_deposit_particles(PartP<T> p, GridP<T> g, int64_t n, double* __restrict__ rho)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int first[3] = {0, 0, 0};
    T wt[3][P + 1];
#pragma unroll
    for (int c = 0; c < D; ++c) {
        T t = grid_coord(p.x[c][i], g.h[c], g.inv_h[c], g.hmul);
        spline_weights<T, P>(t, cell_index(t, g.n[c]), first[c], wt[c]);
    }
    const T q = p.w[i] * g.inv_vol;
    if (D == 2) {
#pragma unroll
        for (int b = 0; b <= P; ++b) {
            const int jy = fold(first[1] + b, g.n[1]);
            const T qy = q * wt[1][b];
#pragma unroll
            for (int a = 0; a <= P; ++a) {
                const int jx = fold(first[0] + a, g.n[0]);
                atomicAdd(&rho[jx + g.n[0] * jy], (double)(qy * wt[0][a]));
            }
        }
    } else {
#pragma unroll
        for (int cz = 0; cz <= P; ++cz) {
            const int jz = fold(first[2] + cz, g.n[2]);
            const T qz = q * wt[2][cz];
#pragma unroll
            for (int b = 0; b <= P; ++b) {
                const int jy = fold(first[1] + b, g.n[1]);
                const T qy = qz * wt[1][b];
                const int64_t row = (int64_t)g.n[0] * (jy + (int64_t)g.n[1] * jz);
#pragma unroll
                for (int a = 0; a <= P; ++a) {
                    const int jx = fold(first[0] + a, g.n[0]);
                    atomicAdd(&rho[row + jx], (double)(qy * wt[0][a]));
                }
            }
        }
    }
}

// rho is accumulated in double (racc): directly in rho for fp64 grids, in the workspace grid for
// fp32 grids, which is then rounded once -- so the fp32 result does not depend on how many
// addends a node receives (clustered config 4) or on the order of the atomics.
template <typename T, int D, int P>
static int deposit_impl(const pic_grid_t& g, const pic_particles_t& p, int order_state, const int32_t* cell_offsets,
                        void* rho, double* racc_ws, cudaStream_t st)
{
    int64_t C = 1;
    for (int c = 0; c < g.dim; ++c) C *= g.n[c];
    double* racc = sizeof(T) == 8 ? (double*)rho : racc_ws;
    if (!racc) return PIC_ERR_WORKSPACE;
    PIC_CUDA_OK(cudaMemsetAsync(racc, 0, sizeof(double) * (size_t)C, st));
    if (p.n > 0) {
        if (order_state != PIC_ORDER_UNSORTED) {       // cell order, exact or stale: runs of equal key (cell_offsets is not read)
            int rc = launch_runs<T, D, P, kModeDeposit, false>(g, p, p, nullptr, nullptr, racc, 0.0, 0.0, st);
            if (rc != PIC_OK) return rc;
        } else {
            k_deposit_particles<T, D, P><<<(unsigned)((p.n + 255) / 256), 256, 0, st>>>(make_partp<T>(p), make_gridp<T>(g),
                                                                                       p.n, racc);
            count_launch();
        }
    }
    if (sizeof(T) == 4) {
        k_round_rho<T><<<(unsigned)((C + 255) / 256), 256, 0, st>>>(racc, (T*)rho, C);
        count_launch();
    }
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

template <typename T, int D>
static int deposit_order(const pic_grid_t& g, const pic_particles_t& p, int order_state, const int32_t* cell_offsets,
                         void* rho, double* racc, cudaStream_t st)
{
    switch (g.order) {
    case 1: return deposit_impl<T, D, 1>(g, p, order_state, cell_offsets, rho, racc, st);
    case 2: return deposit_impl<T, D, 2>(g, p, order_state, cell_offsets, rho, racc, st);
    default: return deposit_impl<T, D, 3>(g, p, order_state, cell_offsets, rho, racc, st);
    }
}

int launch_deposit(const pic_grid_t& g, const pic_particles_t& p, int order_state, const int32_t* cell_offsets,
                   void* rho, double* racc, cudaStream_t st)
{
    if (g.dtype == PIC_F32)
        return g.dim == 2 ? deposit_order<float, 2>(g, p, order_state, cell_offsets, rho, racc, st)
                          : deposit_order<float, 3>(g, p, order_state, cell_offsets, rho, racc, st);
    return g.dim == 2 ? deposit_order<double, 2>(g, p, order_state, cell_offsets, rho, racc, st)
                      : deposit_order<double, 3>(g, p, order_state, cell_offsets, rho, racc, st);
}

}  // namespace pic
