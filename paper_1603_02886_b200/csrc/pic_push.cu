// pic_push.cu -- field gather + accel + push in one pass (rows a6-a7).
//
//   E_i = sum_j E[j] prod_c W_p(x_ic/h_c - j_c)       same splines as the deposit
//   v_i += qm*dt*E_i   (accel, field at the old position)
//   x_i += dt*v_i      (push,  PAPER.md:83, the new velocity), periodic wrap
//
// The paper keeps accel and push apart only because of its grid-vs-particle data view
// and counts 6 loads + 3 stores for each; fused they are
// 2d loads + 2d stores per particle.  k_push_particles reads E through the read-only path
// ("scattered reads through read-only data cache") and is correct for any order.
#include "pic_runs.cuh"

namespace pic {

template <typename T, int D, int P>
__global__ void __launch_bounds__(256) k_push_particles(PartP<T> p, GridP<T> g, FieldP<T> f, int64_t n, double dtd, double qmdtd)
{
    const T dt = (T)dtd, qmdt = (T)qmdtd;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int first[3] = {0, 0, 0};
    T wt[3][P + 1];
    T x[D], v[D], e[D];
#pragma unroll
    for (int c = 0; c < D; ++c) {
        x[c] = p.x[c][i];
        v[c] = p.v[c][i];
        e[c] = (T)0;
        T t = grid_coord(x[c], g.h[c], g.inv_h[c], g.hmul);
        spline_weights<T, P>(t, cell_index(t, g.n[c]), first[c], wt[c]);
    }
    int jx[P + 1];
#pragma unroll
    for (int a = 0; a <= P; ++a) jx[a] = fold(first[0] + a, g.n[0]);
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
                const T wgt = wyz * wt[0][a];
#pragma unroll
                for (int c = 0; c < D; ++c) e[c] += wgt * __ldg(f.E[c] + row + jx[a]);
            }
        }
    }
#pragma unroll
    for (int c = 0; c < D; ++c) {
        const T vn = v[c] + qmdt * e[c];
        T xn = x[c] + dt * vn;
        if (!(xn >= (T)0 && xn < g.L[c])) xn = advance_wrap<T>(x[c], v[c], e[c], dtd, qmdtd, g.Ld[c]);
        p.v[c][i] = vn;
        p.x[c][i] = xn;
    }
}

template <typename T, int D, int P>
static int push_impl(const pic_grid_t& g, pic_particles_t& p, int order_state, const int32_t* cell_offsets,
                     const void* const E[3], double dt, double qm, cudaStream_t st)
{
    if (p.n > 0) {
        if (order_state != PIC_ORDER_UNSORTED)         // cell order, exact or stale: runs of equal key (cell_offsets is not read)
            return launch_runs<T, D, P, kModePush, false>(g, p, p, nullptr, E, nullptr, dt, qm, st);
        FieldP<T> f;
        for (int c = 0; c < 3; ++c) f.E[c] = c < D ? (const T*)E[c] : nullptr;
        k_push_particles<T, D, P><<<(unsigned)((p.n + 255) / 256), 256, 0, st>>>(make_partp<T>(p), make_gridp<T>(g), f, p.n,
                                                                                dt, qm * dt);
        count_launch();
    }
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

template <typename T, int D>
static int push_order(const pic_grid_t& g, pic_particles_t& p, int order_state, const int32_t* cell_offsets,
                      const void* const E[3], double dt, double qm, cudaStream_t st)
{
    switch (g.order) {
    case 1: return push_impl<T, D, 1>(g, p, order_state, cell_offsets, E, dt, qm, st);
    case 2: return push_impl<T, D, 2>(g, p, order_state, cell_offsets, E, dt, qm, st);
    default: return push_impl<T, D, 3>(g, p, order_state, cell_offsets, E, dt, qm, st);
    }
}

int launch_push(const pic_grid_t& g, pic_particles_t& p, int order_state, const int32_t* cell_offsets,
                const void* const E[3], double dt, double qm, cudaStream_t st)
{
    if (g.dtype == PIC_F32)
        return g.dim == 2 ? push_order<float, 2>(g, p, order_state, cell_offsets, E, dt, qm, st)
                          : push_order<float, 3>(g, p, order_state, cell_offsets, E, dt, qm, st);
    return g.dim == 2 ? push_order<double, 2>(g, p, order_state, cell_offsets, E, dt, qm, st)
                      : push_order<double, 3>(g, p, order_state, cell_offsets, E, dt, qm, st);
}

}  // namespace pic
