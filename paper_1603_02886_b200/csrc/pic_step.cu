// pic_step.cu -- the fused kernel of pic_step (row a8): deposit at x(t), gather, accel and push in
// ONE pass over the sorted particles (with perm != NULL also the reorder of the sort, row a4:
// particle perm[j] of src is read, slot j of p is written).  Legal because E is prescribed and frozen ("particles move
// into a frozen given electric field"): rho(x^t) and the push of x^t
// read the same particle data once.  Kernel: k_runs<MODE = deposit|push> (pic_runs.cuh).
#include "pic_runs.cuh"
#include "pic_tile.cuh"

namespace pic {

template <typename T, int D, int P>
static int fused_impl(const pic_grid_t& g, const pic_particles_t& src, pic_particles_t& p, const int32_t* perm,
                      const SortWs& ws, void* rho, const void* const E[3], double dt, double qm, cudaStream_t st, bool cell_sorted,
                      const int32_t* key_offsets)
{
    int64_t C = 1;
    for (int c = 0; c < g.dim; ++c) C *= g.n[c];
    double* racc = sizeof(T) == 8 ? (double*)rho : ws.racc;
    PIC_CUDA_OK(cudaMemsetAsync(racc, 0, sizeof(double) * (size_t)C, st));
    int rc;
    int64_t bucket_cells = 1;
    for (int c = 0; c < g.dim; ++c) bucket_cells *= ws.bucket ? ws.bucket[c] : 1;
    // (small buckets: few tile nodes under many particles, the shared-memory atomics of a warp pile up on the same
    // nodes and the run kernel with strays is faster -- measured crossover near 3^3 cells, profiles/r02_final.md)
    if (perm && !cell_sorted && key_offsets && ws.bucket && bucket_cells >= 27 && tile_bytes<T>(g, ws.bucket) <= kTileMaxBytes) {
        // perm groups the particles by BUCKET (pic_step_buckets) and the bucket's grid tile fits in shared memory: the
        // paper's design, a block per bucket with the tile staged there (pic_tile.cuh).  Same device-side choice between
        // one pass through perm and reorder-then-in-place as below.
        PIC_CUDA_OK(cudaMemsetAsync(ws.chain_sig, 0, sizeof(ChainSig), st));
        rc = launch_bucket_tile<T, D, P, true>(g, ws.bucket, ws.nkeys, src, p, perm, key_offsets, E, racc, dt, qm, st, ws.gate, 0u);
        if (rc != PIC_OK) return rc;
        if ((rc = launch_reorder_records(g, src, p, perm, ws.rec_scratch, ws.gate, 1u, st)) != PIC_OK) return rc;
        rc = launch_bucket_tile<T, D, P, false>(g, ws.bucket, ws.nkeys, p, p, nullptr, key_offsets, E, racc, dt, qm, st, ws.gate, 1u);
        if (rc != PIC_OK) return rc;
    } else if (perm && !cell_sorted) {
        // perm groups the particles by BUCKET (pic_step_buckets): inside a bucket of several cells they keep their
        // source order, so a run of equal cell key is short and most particles are alone in theirs.  The same pass;
        // lone particles are set aside for k_strays (threads on particles, setrho 3.3.4), the others
        // go run by run.  Nothing is emitted (the next sort's key is not the cell key).
        PIC_CUDA_OK(cudaMemsetAsync(ws.chain_sig, 0, sizeof(ChainSig), st));
        PIC_CUDA_OK(cudaMemsetAsync(ws.stray_count, 0, sizeof(uint32_t), st));
        rc = launch_runs<T, D, P, kModeBoth, true>(g, src, p, perm, E, racc, dt, qm, st, ws.gate, 0u, ws.stray_list, ws.stray_count);
        if (rc != PIC_OK) return rc;
        if ((rc = launch_reorder_records(g, src, p, perm, ws.rec_scratch, ws.gate, 1u, st)) != PIC_OK) return rc;
        rc = launch_runs<T, D, P, kModeBoth, false>(g, p, p, nullptr, E, racc, dt, qm, st, ws.gate, 1u, ws.stray_list, ws.stray_count);
        if (rc != PIC_OK) return rc;
        if ((rc = launch_strays<T, D, P, kModeBoth>(g, p, E, racc, dt, qm, ws.stray_list, ws.stray_count, sm_count(), st)) != PIC_OK) return rc;
    } else if (perm) {
        // steady state: ONE pass through perm.  Most particles moving (first step, garbage hint): the scattered
        // gather is done by the high-occupancy reorder kernel first and the pass runs in place.  *ws.gate, written
        // by the sort, selects on the device: the kernels of the other arm return at once.  Either way the pass
        // leaves the next sort's inputs behind (EmitP): the counters it adds to are zero from here on.
        PIC_CUDA_OK(cudaMemsetAsync(ws.emit_begin, 0, ws.emit_bytes, st));
        rc = launch_runs<T, D, P, kModeBoth, true>(g, src, p, perm, E, racc, dt, qm, st, ws.gate, 0u, nullptr, nullptr, &ws.emit);
        if (rc != PIC_OK) return rc;
        if ((rc = launch_reorder_records(g, src, p, perm, ws.rec_scratch, ws.gate, 1u, st)) != PIC_OK) return rc;
        rc = launch_runs<T, D, P, kModeBoth, false>(g, p, p, nullptr, E, racc, dt, qm, st, ws.gate, 1u, nullptr, nullptr, &ws.emit);
        if (rc != PIC_OK) return rc;
        if (p.n > 0 && (rc = launch_chain_commit(g, p, ws, st)) != PIC_OK) return rc;
    } else {
        // the order of an earlier sort, in place: lone particles (drifted since) are set aside for k_strays.  The
        // positions change under the workspace's emission, if any: it is void from here on
        PIC_CUDA_OK(cudaMemsetAsync(ws.chain_sig, 0, sizeof(ChainSig), st));
        PIC_CUDA_OK(cudaMemsetAsync(ws.stray_count, 0, sizeof(uint32_t), st));
        rc = launch_runs<T, D, P, kModeBoth, false>(g, p, p, nullptr, E, racc, dt, qm, st, nullptr, 0u, ws.stray_list, ws.stray_count);
        if (rc != PIC_OK) return rc;
        if ((rc = launch_strays<T, D, P, kModeBoth>(g, p, E, racc, dt, qm, ws.stray_list, ws.stray_count, sm_count(), st)) != PIC_OK) return rc;
    }
    if (sizeof(T) == 4) {
        k_round_rho<T><<<(unsigned)((C + 255) / 256), 256, 0, st>>>(racc, (T*)rho, C);
        count_launch();
    }
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

template <typename T, int D>
static int fused_order(const pic_grid_t& g, const pic_particles_t& src, pic_particles_t& p, const int32_t* perm,
                       const SortWs& ws, void* rho, const void* const E[3], double dt, double qm, cudaStream_t st, bool cell_sorted,
                       const int32_t* key_offsets)
{
    switch (g.order) {
    case 1: return fused_impl<T, D, 1>(g, src, p, perm, ws, rho, E, dt, qm, st, cell_sorted, key_offsets);
    case 2: return fused_impl<T, D, 2>(g, src, p, perm, ws, rho, E, dt, qm, st, cell_sorted, key_offsets);
    default: return fused_impl<T, D, 3>(g, src, p, perm, ws, rho, E, dt, qm, st, cell_sorted, key_offsets);
    }
}

// The closed loop (PAPER.md:79-84 steps i-iv with the field solve in): rho at x(t) while the
// particles are reordered (one pass along perm), field_solver, then accel + push in place with the new field.
template <typename T, int D, int P>
static int selfconsistent_impl(const pic_grid_t& g, const pic_particles_t& src, pic_particles_t& p, const int32_t* perm,
                               const SortWs& ws, void* rho, void* const E[3], void* field_ws, double dt, double qm, cudaStream_t st)
{
    int64_t C = 1;
    for (int c = 0; c < g.dim; ++c) C *= g.n[c];
    double* racc = sizeof(T) == 8 ? (double*)rho : ws.racc;
    PIC_CUDA_OK(cudaMemsetAsync(racc, 0, sizeof(double) * (size_t)C, st));
    PIC_CUDA_OK(cudaMemsetAsync(ws.chain_sig, 0, sizeof(ChainSig), st));       // nothing is emitted: no chain from here
    int rc = launch_runs<T, D, P, kModeDeposit, true>(g, src, p, perm, nullptr, racc, 0.0, 0.0, st, ws.gate, 0u);
    if (rc != PIC_OK) return rc;
    if ((rc = launch_reorder_records(g, src, p, perm, ws.rec_scratch, ws.gate, 1u, st)) != PIC_OK) return rc;
    if ((rc = launch_runs<T, D, P, kModeDeposit, false>(g, p, p, nullptr, nullptr, racc, 0.0, 0.0, st, ws.gate, 1u)) != PIC_OK) return rc;
    if (sizeof(T) == 4) {
        k_round_rho<T><<<(unsigned)((C + 255) / 256), 256, 0, st>>>(racc, (T*)rho, C);
        count_launch();
    }
    mark_phase(PIC_PHASE_DEPOSIT, st);
    if ((rc = launch_field_solve(g, rho, E, nullptr, field_ws, st)) != PIC_OK) return rc;
    const void* Ec[3] = {E[0], E[1], E[2]};
    return launch_runs<T, D, P, kModePush, false>(g, p, p, nullptr, Ec, nullptr, dt, qm, st);
}

template <typename T, int D>
static int selfconsistent_order(const pic_grid_t& g, const pic_particles_t& src, pic_particles_t& p, const int32_t* perm,
                                const SortWs& ws, void* rho, void* const E[3], void* field_ws, double dt, double qm, cudaStream_t st)
{
    switch (g.order) {
    case 1: return selfconsistent_impl<T, D, 1>(g, src, p, perm, ws, rho, E, field_ws, dt, qm, st);
    case 2: return selfconsistent_impl<T, D, 2>(g, src, p, perm, ws, rho, E, field_ws, dt, qm, st);
    default: return selfconsistent_impl<T, D, 3>(g, src, p, perm, ws, rho, E, field_ws, dt, qm, st);
    }
}

int launch_selfconsistent(const pic_grid_t& g, const pic_particles_t& src, pic_particles_t& p, const int32_t* perm,
                          const SortWs& ws, void* rho, void* const E[3], void* field_ws, double dt, double qm, cudaStream_t st)
{
    if (g.dtype == PIC_F32)
        return g.dim == 2 ? selfconsistent_order<float, 2>(g, src, p, perm, ws, rho, E, field_ws, dt, qm, st)
                          : selfconsistent_order<float, 3>(g, src, p, perm, ws, rho, E, field_ws, dt, qm, st);
    return g.dim == 2 ? selfconsistent_order<double, 2>(g, src, p, perm, ws, rho, E, field_ws, dt, qm, st)
                      : selfconsistent_order<double, 3>(g, src, p, perm, ws, rho, E, field_ws, dt, qm, st);
}

int launch_fused(const pic_grid_t& g, const pic_particles_t& src, pic_particles_t& p, const int32_t* perm,
                 const SortWs& ws, void* rho, const void* const E[3], double dt, double qm, cudaStream_t st, bool cell_sorted,
                 const int32_t* key_offsets)
{
    if (g.dtype == PIC_F32)
        return g.dim == 2 ? fused_order<float, 2>(g, src, p, perm, ws, rho, E, dt, qm, st, cell_sorted, key_offsets)
                          : fused_order<float, 3>(g, src, p, perm, ws, rho, E, dt, qm, st, cell_sorted, key_offsets);
    return g.dim == 2 ? fused_order<double, 2>(g, src, p, perm, ws, rho, E, dt, qm, st, cell_sorted, key_offsets)
                      : fused_order<double, 3>(g, src, p, perm, ws, rho, E, dt, qm, st, cell_sorted, key_offsets);
}

}  // namespace pic
