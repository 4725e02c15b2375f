// pic_step.cu -- the fused kernel of pic_step (row a8): deposit at x(t), gather, accel and push in
// ONE pass over the sorted particles (with perm != NULL also the reorder of the sort, row a4:
// particle perm[j] of src is read, slot j of p is written).  Legal because E is prescribed and frozen ("particles move
// into a frozen given electric field"): rho(x^t) and the push of x^t
// read the same particle data once.  Kernel: k_rows<MODE = deposit|push> (pic_rows.cuh).
#include <cstdlib>

#include "pic_rows.cuh"
#include "pic_runs.cuh"

namespace pic {

template <typename T, int D, int P>
static int fused_impl(const pic_grid_t& g, const pic_particles_t& src, pic_particles_t& p, const int32_t* perm,
                      const int32_t* cell_offsets, void* rho, const void* const E[3], double dt, double qm,
                      double* racc_ws, cudaStream_t st)
{
    int64_t C = 1;
    for (int c = 0; c < g.dim; ++c) C *= g.n[c];
    double* racc = sizeof(T) == 8 ? (double*)rho : racc_ws;
    if (!racc) return PIC_ERR_WORKSPACE;
    PIC_CUDA_OK(cudaMemsetAsync(racc, 0, sizeof(double) * (size_t)C, st));
    static const bool old_kernel = getenv("PIC_OLD_ROWS") != nullptr;      // TEMP: A/B switch
    int rc;
    if (old_kernel)
        rc = perm ? launch_rows<T, D, P, kModeBoth, true>(g, src, p, perm, cell_offsets, E, racc, dt, qm, st)
                  : launch_rows<T, D, P, kModeBoth, false>(g, p, p, nullptr, cell_offsets, E, racc, dt, qm, st);
    else
        rc = perm ? launch_runs<T, D, P, kModeBoth, true>(g, src, p, perm, E, racc, dt, qm, st)
                  : launch_runs<T, D, P, kModeBoth, false>(g, p, p, nullptr, E, racc, dt, qm, st);
    if (rc != PIC_OK) return rc;
    if (sizeof(T) == 4) {
        k_round_rho<T><<<(unsigned)((C + 255) / 256), 256, 0, st>>>(racc, (T*)rho, C);
        count_launch();
    }
    return cudaGetLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

template <typename T, int D>
static int fused_order(const pic_grid_t& g, const pic_particles_t& src, pic_particles_t& p, const int32_t* perm,
                       const int32_t* cell_offsets, void* rho, const void* const E[3], double dt, double qm,
                       double* racc, cudaStream_t st)
{
    switch (g.order) {
    case 1: return fused_impl<T, D, 1>(g, src, p, perm, cell_offsets, rho, E, dt, qm, racc, st);
    case 2: return fused_impl<T, D, 2>(g, src, p, perm, cell_offsets, rho, E, dt, qm, racc, st);
    default: return fused_impl<T, D, 3>(g, src, p, perm, cell_offsets, rho, E, dt, qm, racc, st);
    }
}

template <typename T, int D, int P>
static int stale_impl(const pic_grid_t& g, pic_particles_t& p, const int32_t* cell_offsets, void* rho, const void* const E[3],
                      double dt, double qm, double* racc_ws, uint32_t* gate, cudaStream_t st)
{
    int64_t C = 1;
    for (int c = 0; c < g.dim; ++c) C *= g.n[c];
    double* racc = sizeof(T) == 8 ? (double*)rho : racc_ws;
    if (!racc) return PIC_ERR_WORKSPACE;
    int rc = launch_offsets_check(g, cell_offsets, p.n, gate, st);
    if (rc != PIC_OK) return rc;
    PIC_CUDA_OK(cudaMemsetAsync(racc, 0, sizeof(double) * (size_t)C, st));
    // offsets usable: one pass, cell by cell; particles that left their cell take the out-of-line path
    rc = launch_rows<T, D, P, kModeBoth, false>(g, p, p, nullptr, cell_offsets, E, racc, dt, qm, st, gate, 0u);
    if (rc != PIC_OK) return rc;
    mark_phase(PIC_PHASE_DEPOSIT, st);
    // offsets not usable: threads on particles (setrho 3.3.4), deposit at x(t) before the push
    if ((rc = launch_deposit_particles(g, p, racc, gate, 1u, st)) != PIC_OK) return rc;
    if (sizeof(T) == 4) {
        k_round_rho<T><<<(unsigned)((C + 255) / 256), 256, 0, st>>>(racc, (T*)rho, C);
        count_launch();
    }
    return launch_push_particles(g, p, E, dt, qm, gate, 1u, st);
}

template <typename T, int D>
static int stale_order(const pic_grid_t& g, pic_particles_t& p, const int32_t* cell_offsets, void* rho, const void* const E[3],
                       double dt, double qm, double* racc, uint32_t* gate, cudaStream_t st)
{
    switch (g.order) {
    case 1: return stale_impl<T, D, 1>(g, p, cell_offsets, rho, E, dt, qm, racc, gate, st);
    case 2: return stale_impl<T, D, 2>(g, p, cell_offsets, rho, E, dt, qm, racc, gate, st);
    default: return stale_impl<T, D, 3>(g, p, cell_offsets, rho, E, dt, qm, racc, gate, st);
    }
}

int launch_stale_step(const pic_grid_t& g, pic_particles_t& p, const int32_t* cell_offsets, void* rho,
                      const void* const E[3], double dt, double qm, double* racc, uint32_t* gate, cudaStream_t st)
{
    if (g.dtype == PIC_F32)
        return g.dim == 2 ? stale_order<float, 2>(g, p, cell_offsets, rho, E, dt, qm, racc, gate, st)
                          : stale_order<float, 3>(g, p, cell_offsets, rho, E, dt, qm, racc, gate, st);
    return g.dim == 2 ? stale_order<double, 2>(g, p, cell_offsets, rho, E, dt, qm, racc, gate, st)
                      : stale_order<double, 3>(g, p, cell_offsets, rho, E, dt, qm, racc, gate, st);
}

int launch_fused(const pic_grid_t& g, const pic_particles_t& src, pic_particles_t& p, const int32_t* perm,
                 const int32_t* cell_offsets, void* rho, const void* const E[3], double dt, double qm, double* racc,
                 cudaStream_t st)
{
    if (g.dtype == PIC_F32)
        return g.dim == 2 ? fused_order<float, 2>(g, src, p, perm, cell_offsets, rho, E, dt, qm, racc, st)
                          : fused_order<float, 3>(g, src, p, perm, cell_offsets, rho, E, dt, qm, racc, st);
    return g.dim == 2 ? fused_order<double, 2>(g, src, p, perm, cell_offsets, rho, E, dt, qm, racc, st)
                      : fused_order<double, 3>(g, src, p, perm, cell_offsets, rho, E, dt, qm, racc, st);
}

}  // namespace pic
