// pic_api.cu -- the extern "C" entry points declared in include/pic.h: argument validation,
// workspace carving, and the order of kernel launches.  No arithmetic of the method lives here.
#include <cstring>

#include "pic_common.cuh"

namespace pic {

static thread_local int g_launches = 0;
void count_launch(int n) { g_launches += n; }

int sm_count()
{
    // asked several times per step: the attribute query is made once per device (a benign race: every thread that
    // loses it writes the same number)
    static int cached[64] = {};
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 148;
    if (dev >= 0 && dev < 64 && cached[dev] > 0) return cached[dev];
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) return 148;
    if (dev >= 0 && dev < 64) cached[dev] = sms;
    return sms;
}

static thread_local cudaEvent_t g_events[PIC_NUM_PHASES];
static thread_local int g_num_events = 0;
void mark_phase(int phase, cudaStream_t st)
{
    if (phase < g_num_events && g_events[phase]) cudaEventRecord(g_events[phase], st);
}

static inline size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

static bool aligned16(const void* p) { return p != nullptr && ((uintptr_t)p & 15u) == 0; }

static int64_t cells_of(const pic_grid_t& g)
{
    int64_t C = 1;
    for (int c = 0; c < g.dim; ++c) C *= g.n[c];
    return C;
}

static int check_grid(const pic_grid_t* g)
{
    if (!g) return PIC_ERR_INVALID_ARG;
    if (g->dim != 2 && g->dim != 3) return PIC_ERR_INVALID_ARG;
    if (g->order < 1 || g->order > 3) return PIC_ERR_INVALID_ARG;
    if (g->dtype != PIC_F32 && g->dtype != PIC_F64) return PIC_ERR_INVALID_ARG;
    int64_t C = 1;
    for (int c = 0; c < g->dim; ++c) {
        if (g->n[c] < g->order + 1) return PIC_ERR_INVALID_ARG;   // a stencil must not wrap onto itself
        if (!(g->h[c] > 0.0) || !(g->h[c] < 1e300)) return PIC_ERR_INVALID_ARG;
        C *= g->n[c];
        if (C >= ((int64_t)1 << 31)) return PIC_ERR_INVALID_ARG;
    }
    return PIC_OK;
}

// n_override >= 0: p is an OUTPUT set whose own n is not read (it receives n_override particles)
static int check_particles(const pic_grid_t& g, const pic_particles_t* p, bool need_v, bool need_w, int64_t n_override = -1)
{
    if (!p) return PIC_ERR_INVALID_ARG;
    const int64_t n = n_override >= 0 ? n_override : p->n;
    if (n < 0 || n >= ((int64_t)1 << 30)) return PIC_ERR_INVALID_ARG;
    if (n == 0) return PIC_OK;                         // empty arrays may be null
    for (int c = 0; c < g.dim; ++c) {
        if (!aligned16(p->x[c])) return PIC_ERR_INVALID_ARG;
        if (need_v && !aligned16(p->v[c])) return PIC_ERR_INVALID_ARG;
    }
    if (need_w && !aligned16(p->w)) return PIC_ERR_INVALID_ARG;
    return PIC_OK;
}

// does any array of a overlap any array of b (n elements each)?
static bool aliases(const pic_grid_t& g, const pic_particles_t& a, const pic_particles_t& b, int64_t n)
{
    const char* pa[7];
    const char* pb[7];
    int m = 0;
    for (int c = 0; c < g.dim; ++c) {
        pa[m] = (const char*)a.x[c]; pb[m++] = (const char*)b.x[c];
        pa[m] = (const char*)a.v[c]; pb[m++] = (const char*)b.v[c];
    }
    pa[m] = (const char*)a.w; pb[m++] = (const char*)b.w;
    const size_t bytes = (size_t)n * (g.dtype == PIC_F64 ? 8 : 4);
    for (int i = 0; i < m; ++i)
        for (int j = 0; j < m; ++j)
            if (pa[i] < pb[j] + bytes && pb[j] < pa[i] + bytes) return true;
    return false;
}

// A call that uses a workspace for anything but a chained step ends the chain a previous pic_step may have left in
// it (PIC_SORT_CHAINED): the signature sits in the first bytes of every workspace layout, whatever n and the grid are.
static int void_chain(void* ws, cudaStream_t st)
{
    static_assert(sizeof(ChainSig) <= 256, "the signature has the first 256 bytes of the workspace");
    return cudaMemsetAsync(ws, 0, sizeof(ChainSig), st) == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

static int check_bucket(const pic_grid_t& g, const int32_t* bucket)
{
    if (!bucket) return PIC_ERR_INVALID_ARG;
    for (int c = 0; c < g.dim; ++c)
        if (bucket[c] < 1 || bucket[c] > g.n[c]) return PIC_ERR_INVALID_ARG;
    return PIC_OK;
}

static int check_field(const pic_grid_t& g, const void* const E[3])
{
    if (!E) return PIC_ERR_INVALID_ARG;
    for (int c = 0; c < g.dim; ++c)
        if (!aligned16(E[c])) return PIC_ERR_INVALID_ARG;
    return PIC_OK;
}

}  // namespace pic

using namespace pic;

extern "C" {

int pic_last_launch_count(void) { return g_launches; }

int pic_set_phase_events(void* const* events, int count)
{
    if (count < 0 || count > PIC_NUM_PHASES || (count > 0 && !events)) return PIC_ERR_INVALID_ARG;
    g_num_events = count;
    for (int k = 0; k < count; ++k) g_events[k] = (cudaEvent_t)events[k];
    return PIC_OK;
}

const char* pic_strerror(int status)
{
    switch (status) {
    case PIC_OK: return "ok";
    case PIC_ERR_INVALID_ARG: return "invalid argument";
    case PIC_ERR_UNSUPPORTED: return "unsupported configuration";
    case PIC_ERR_WORKSPACE: return "workspace too small";
    case PIC_ERR_CUDA: return "CUDA launch or runtime failure";
    case PIC_ERR_TOO_LARGE: return "grid has more nodes than the library's static scratch array (PIC_DEPOSIT_STATIC_MAX_NODES)";
    default: return "unknown status";
    }
}

int pic_workspace_bytes(const pic_grid_t* grid, int64_t n, size_t* bytes)
{
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if (!bytes || n < 0 || n >= ((int64_t)1 << 30)) return PIC_ERR_INVALID_ARG;
    *bytes = sort_ws_bytes(*grid, n);
    return PIC_OK;
}

int pic_sort(const pic_grid_t* grid, const pic_particles_t* in, pic_particles_t* out, int32_t* perm,
             int32_t* cell_offsets, void* ws, size_t ws_bytes, void* stream)
{
    g_launches = 0;
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if ((rc = check_particles(*grid, in, true, true)) != PIC_OK) return rc;
    if ((rc = check_particles(*grid, out, true, true, in->n)) != PIC_OK) return rc;
    if ((in->n > 0 && !aligned16(perm)) || !aligned16(cell_offsets) || !aligned16(ws)) return PIC_ERR_INVALID_ARG;
    if (in->n > 0 && aliases(*grid, *in, *out, in->n)) return PIC_ERR_INVALID_ARG;
    SortWs sws;
    if ((rc = carve_sort_ws(*grid, in->n, ws, ws_bytes, sws)) != PIC_OK) return rc;
    pic_particles_t o = *out;
    o.n = in->n;
    return launch_sort(*grid, *in, o, perm, cell_offsets, sws, true, false, (cudaStream_t)stream);
}

int pic_deposit(const pic_grid_t* grid, const pic_particles_t* p, int order_state, const int32_t* cell_offsets,
                void* rho, void* ws, size_t ws_bytes, void* stream)
{
    g_launches = 0;
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if ((rc = check_particles(*grid, p, false, true)) != PIC_OK) return rc;
    double* racc = nullptr;
    if (grid->dtype == PIC_F32) {          // fp32 grids accumulate in a double grid of the workspace
        if (!aligned16(ws)) return PIC_ERR_INVALID_ARG;
        SortWs sws;
        if ((rc = carve_sort_ws(*grid, p->n, ws, ws_bytes, sws)) != PIC_OK) return rc;
        racc = sws.racc;
    }
    if (order_state < PIC_ORDER_UNSORTED || order_state > PIC_ORDER_STALE) return PIC_ERR_INVALID_ARG;
    if (order_state != PIC_ORDER_UNSORTED && !aligned16(cell_offsets)) return PIC_ERR_INVALID_ARG;
    if (!aligned16(rho)) return PIC_ERR_INVALID_ARG;
    if (racc && (rc = void_chain(ws, (cudaStream_t)stream)) != PIC_OK) return rc;     // the workspace is written: no chain from here
    mark_phase(PIC_PHASE_BEGIN, (cudaStream_t)stream);
    rc = launch_deposit(*grid, *p, order_state, cell_offsets, rho, racc, (cudaStream_t)stream);
    mark_phase(PIC_PHASE_DEPOSIT, (cudaStream_t)stream);
    return rc;
}

int pic_deposit_nodes(const pic_grid_t* grid, const pic_particles_t* p, const int32_t* cell_offsets, void* rho, void* ws,
                      size_t ws_bytes, void* stream)
{
    g_launches = 0;
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if ((rc = check_particles(*grid, p, false, true)) != PIC_OK) return rc;
    if (!aligned16(cell_offsets) || !aligned16(rho) || !aligned16(ws)) return PIC_ERR_INVALID_ARG;
    SortWs sws;
    if ((rc = carve_sort_ws(*grid, p->n, ws, ws_bytes, sws)) != PIC_OK) return rc;
    if ((rc = void_chain(ws, (cudaStream_t)stream)) != PIC_OK) return rc;
    mark_phase(PIC_PHASE_BEGIN, (cudaStream_t)stream);
    rc = launch_deposit_nodes(*grid, *p, cell_offsets, rho, sws, (cudaStream_t)stream);
    mark_phase(PIC_PHASE_DEPOSIT, (cudaStream_t)stream);
    return rc;
}

int pic_deposit_replicated_bytes(const pic_grid_t* grid, int64_t n, size_t* bytes)
{
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if (!bytes || n < 0 || n >= ((int64_t)1 << 30)) return PIC_ERR_INVALID_ARG;
    *bytes = sort_ws_bytes(*grid, n) + replicated_slab_bytes(*grid);
    return PIC_OK;
}

int pic_deposit_replicated(const pic_grid_t* grid, const pic_particles_t* p, const int32_t* cell_offsets, void* rho, void* ws,
                           size_t ws_bytes, void* stream)
{
    g_launches = 0;
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if ((rc = check_particles(*grid, p, false, true)) != PIC_OK) return rc;
    if (!aligned16(cell_offsets) || !aligned16(rho) || !aligned16(ws)) return PIC_ERR_INVALID_ARG;
    const size_t sb = sort_ws_bytes(*grid, p->n);
    if (ws_bytes < sb + replicated_slab_bytes(*grid)) return PIC_ERR_WORKSPACE;
    SortWs sws;
    if ((rc = carve_sort_ws(*grid, p->n, ws, sb, sws)) != PIC_OK) return rc;
    if ((rc = void_chain(ws, (cudaStream_t)stream)) != PIC_OK) return rc;
    mark_phase(PIC_PHASE_BEGIN, (cudaStream_t)stream);
    rc = launch_deposit_replicated(*grid, *p, cell_offsets, rho, sws, (char*)ws + sb, (cudaStream_t)stream);
    mark_phase(PIC_PHASE_DEPOSIT, (cudaStream_t)stream);
    return rc;
}

int pic_push(const pic_grid_t* grid, pic_particles_t* p, int order_state, const int32_t* cell_offsets,
             const void* const E[3], double dt, double qm, void* stream)
{
    g_launches = 0;
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if ((rc = check_particles(*grid, p, true, false)) != PIC_OK) return rc;
    if (order_state < PIC_ORDER_UNSORTED || order_state > PIC_ORDER_STALE) return PIC_ERR_INVALID_ARG;
    if (order_state != PIC_ORDER_UNSORTED && !aligned16(cell_offsets)) return PIC_ERR_INVALID_ARG;
    if ((rc = check_field(*grid, E)) != PIC_OK) return rc;
    mark_phase(PIC_PHASE_BEGIN, (cudaStream_t)stream);
    rc = launch_push(*grid, *p, order_state, cell_offsets, E, dt, qm, (cudaStream_t)stream);
    mark_phase(PIC_PHASE_PUSH, (cudaStream_t)stream);
    return rc;
}

int pic_step(const pic_grid_t* grid, const pic_particles_t* in, pic_particles_t* out, int32_t* perm,
             int32_t* cell_offsets, void* rho, const void* const E[3], double dt, double qm, int do_sort, void* ws,
             size_t ws_bytes, void* stream)
{
    g_launches = 0;
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    // any non-zero value asks for a sort (the ABI of SURVEY 8(b)); PIC_SORT_CHAINED alone asks for the chained one
    const bool chained = do_sort == PIC_SORT_CHAINED;
    if ((rc = check_particles(*grid, in, true, true)) != PIC_OK) return rc;
    if ((rc = check_particles(*grid, out, true, true, in->n)) != PIC_OK) return rc;
    if ((rc = check_field(*grid, E)) != PIC_OK) return rc;
    if (!aligned16(rho)) return PIC_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    pic_particles_t o = *out;
    o.n = in->n;
    const size_t s = grid->dtype == PIC_F64 ? 8 : 4;
    if (!aligned16(ws)) return PIC_ERR_INVALID_ARG;
    SortWs sws;
    if ((rc = carve_sort_ws(*grid, in->n, ws, ws_bytes, sws)) != PIC_OK) return rc;
    // every argument is checked before the first copy or launch is enqueued
    if (do_sort) {
        if ((in->n > 0 && !aligned16(perm)) || !aligned16(cell_offsets)) return PIC_ERR_INVALID_ARG;
        if (in->n > 0 && aliases(*grid, *in, *out, in->n)) return PIC_ERR_INVALID_ARG;
    } else if (cell_offsets && in->n > 0 && !aligned16(cell_offsets)) {
        return PIC_ERR_INVALID_ARG;
    }
    if (do_sort) {
        // perm and cell_offsets only: the reorder itself happens inside the fused kernel below
        if ((rc = launch_sort(*grid, *in, o, perm, cell_offsets, sws, false, chained, st)) != PIC_OK) return rc;
    } else {
        // keep the current order; out may be the same arrays as in (in-place step)
        for (int c = 0; c < grid->dim; ++c) {
            if (in->x[c] != o.x[c]) PIC_CUDA_OK(cudaMemcpyAsync(o.x[c], in->x[c], s * (size_t)in->n, cudaMemcpyDeviceToDevice, st));
            if (in->v[c] != o.v[c]) PIC_CUDA_OK(cudaMemcpyAsync(o.v[c], in->v[c], s * (size_t)in->n, cudaMemcpyDeviceToDevice, st));
        }
        if (in->w != o.w) PIC_CUDA_OK(cudaMemcpyAsync(o.w, in->w, s * (size_t)in->n, cudaMemcpyDeviceToDevice, st));
    }
    if (!do_sort) mark_phase(PIC_PHASE_BEGIN, st);
    if (do_sort) {                               // one fused kernel over the sorted particles
        rc = launch_fused(*grid, *in, o, perm, sws, rho, E, dt, qm, st);
        mark_phase(PIC_PHASE_PUSH, st);
        return rc;
    }
    if (cell_offsets && in->n > 0) {
        // the order of an earlier sort: the same kernel in place.  It finds the runs of equal cell key itself
        // (cell_offsets is not read), so the result is exact however far the particles have drifted
        rc = launch_fused(*grid, o, o, nullptr, sws, rho, E, dt, qm, st);
        mark_phase(PIC_PHASE_PUSH, st);
        return rc;
    }
    PIC_CUDA_OK(cudaMemsetAsync(sws.chain_sig, 0, sizeof(ChainSig), st));       // positions change: no chain from here
    if ((rc = launch_deposit(*grid, o, PIC_ORDER_UNSORTED, nullptr, rho, sws.racc, st)) != PIC_OK) return rc;
    mark_phase(PIC_PHASE_DEPOSIT, st);
    rc = launch_push(*grid, o, PIC_ORDER_UNSORTED, nullptr, E, dt, qm, st);
    mark_phase(PIC_PHASE_PUSH, st);
    return rc;
}

// ---- buckets of several cells (NEXT-2) -------------------------------------------------------
int pic_bucket_count(const pic_grid_t* grid, const int32_t bucket[3], int64_t* count)
{
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if ((rc = check_bucket(*grid, bucket)) != PIC_OK) return rc;
    if (!count) return PIC_ERR_INVALID_ARG;
    int64_t B = 1;
    for (int c = 0; c < grid->dim; ++c) B *= (grid->n[c] + bucket[c] - 1) / bucket[c];
    *count = B;
    return PIC_OK;
}

int pic_sort_buckets(const pic_grid_t* grid, const int32_t bucket[3], const pic_particles_t* in, pic_particles_t* out,
                     int32_t* perm, int32_t* bucket_offsets, void* ws, size_t ws_bytes, void* stream)
{
    g_launches = 0;
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if ((rc = check_bucket(*grid, bucket)) != PIC_OK) return rc;
    if ((rc = check_particles(*grid, in, true, true)) != PIC_OK) return rc;
    if ((rc = check_particles(*grid, out, true, true, in->n)) != PIC_OK) return rc;
    if ((in->n > 0 && !aligned16(perm)) || !aligned16(bucket_offsets) || !aligned16(ws)) return PIC_ERR_INVALID_ARG;
    if (in->n > 0 && aliases(*grid, *in, *out, in->n)) return PIC_ERR_INVALID_ARG;
    SortWs sws;
    if ((rc = carve_sort_ws(*grid, in->n, ws, ws_bytes, sws, bucket)) != PIC_OK) return rc;
    pic_particles_t o = *out;
    o.n = in->n;
    return launch_sort(*grid, *in, o, perm, bucket_offsets, sws, true, false, (cudaStream_t)stream);
}

int pic_sort_buckets_inplace_bytes(const pic_grid_t* grid, int64_t n, size_t* bytes)
{
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if (!bytes || n < 0 || n >= ((int64_t)1 << 30)) return PIC_ERR_INVALID_ARG;
    const size_t s = grid->dtype == PIC_F64 ? 8 : 4;
    *bytes = sort_ws_bytes(*grid, n) + align256(s * (size_t)(2 * grid->dim + 1) * (size_t)(n > 0 ? n : 1));
    return PIC_OK;
}

int pic_sort_buckets_inplace(const pic_grid_t* grid, const int32_t bucket[3], pic_particles_t* p, int32_t* bucket_offsets,
                             int32_t* moved, void* ws, size_t ws_bytes, void* stream)
{
    g_launches = 0;
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if ((rc = check_bucket(*grid, bucket)) != PIC_OK) return rc;
    if ((rc = check_particles(*grid, p, true, true)) != PIC_OK) return rc;
    if (!aligned16(bucket_offsets) || !aligned16(ws)) return PIC_ERR_INVALID_ARG;
    const size_t s = grid->dtype == PIC_F64 ? 8 : 4;
    const size_t sb = sort_ws_bytes(*grid, p->n);
    if (ws_bytes < sb + align256(s * (size_t)(2 * grid->dim + 1) * (size_t)(p->n > 0 ? p->n : 1))) return PIC_ERR_WORKSPACE;
    SortWs sws;
    if ((rc = carve_sort_ws(*grid, p->n, ws, sb, sws, bucket)) != PIC_OK) return rc;
    return launch_sort_inplace(*grid, *p, bucket_offsets, sws, (char*)ws + sb, moved, (cudaStream_t)stream);
}

int pic_step_buckets(const pic_grid_t* grid, const int32_t bucket[3], const pic_particles_t* in, pic_particles_t* out,
                     int32_t* perm, int32_t* bucket_offsets, void* rho, const void* const E[3], double dt, double qm,
                     void* ws, size_t ws_bytes, void* stream)
{
    g_launches = 0;
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if ((rc = check_bucket(*grid, bucket)) != PIC_OK) return rc;
    if ((rc = check_particles(*grid, in, true, true)) != PIC_OK) return rc;
    if ((rc = check_particles(*grid, out, true, true, in->n)) != PIC_OK) return rc;
    if ((rc = check_field(*grid, E)) != PIC_OK) return rc;
    if (!aligned16(rho) || !aligned16(ws)) return PIC_ERR_INVALID_ARG;
    if ((in->n > 0 && !aligned16(perm)) || !aligned16(bucket_offsets)) return PIC_ERR_INVALID_ARG;
    if (in->n > 0 && aliases(*grid, *in, *out, in->n)) return PIC_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    SortWs sws;
    if ((rc = carve_sort_ws(*grid, in->n, ws, ws_bytes, sws, bucket)) != PIC_OK) return rc;
    pic_particles_t o = *out;
    o.n = in->n;
    if ((rc = launch_sort(*grid, *in, o, perm, bucket_offsets, sws, false, false, st)) != PIC_OK) return rc;
    bool unit = true;                            // one cell per bucket: this is pic_step(PIC_SORT)
    for (int c = 0; c < grid->dim; ++c) unit = unit && bucket[c] == 1;
    rc = launch_fused(*grid, *in, o, perm, sws, rho, E, dt, qm, st, unit, bucket_offsets);
    mark_phase(PIC_PHASE_PUSH, st);
    return rc;
}

// ---- field solve and the closed loop (NEXT-4) -------------------------------------------------
int pic_field_solve_bytes(const pic_grid_t* grid, size_t* bytes)
{
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if (!bytes) return PIC_ERR_INVALID_ARG;
    if ((rc = field_supported(*grid)) != PIC_OK) return rc;
    *bytes = field_ws_bytes(*grid);
    return PIC_OK;
}

int pic_field_solve(const pic_grid_t* grid, const void* rho, void* const E[3], void* phi, void* ws, size_t ws_bytes, void* stream)
{
    g_launches = 0;
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if (!aligned16(rho) || !E || !aligned16(ws) || (phi && !aligned16(phi))) return PIC_ERR_INVALID_ARG;
    for (int c = 0; c < grid->dim; ++c)
        if (!aligned16(E[c])) return PIC_ERR_INVALID_ARG;
    if ((rc = field_supported(*grid)) != PIC_OK) return rc;          // before anything is enqueued
    if (ws_bytes < field_ws_bytes(*grid)) return PIC_ERR_WORKSPACE;
    return launch_field_solve(*grid, rho, E, phi, ws, (cudaStream_t)stream);
}

int pic_step_selfconsistent_bytes(const pic_grid_t* grid, int64_t n, size_t* bytes)
{
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if (!bytes || n < 0 || n >= ((int64_t)1 << 30)) return PIC_ERR_INVALID_ARG;
    if ((rc = field_supported(*grid)) != PIC_OK) return rc;
    *bytes = sort_ws_bytes(*grid, n) + field_ws_bytes(*grid);
    return PIC_OK;
}

int pic_step_selfconsistent(const pic_grid_t* grid, const pic_particles_t* in, pic_particles_t* out, int32_t* perm,
                            int32_t* cell_offsets, void* rho, void* const E[3], double dt, double qm, void* ws,
                            size_t ws_bytes, void* stream)
{
    g_launches = 0;
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if ((rc = check_particles(*grid, in, true, true)) != PIC_OK) return rc;
    if ((rc = check_particles(*grid, out, true, true, in->n)) != PIC_OK) return rc;
    if (!E || !aligned16(rho) || !aligned16(ws)) return PIC_ERR_INVALID_ARG;
    for (int c = 0; c < grid->dim; ++c)
        if (!aligned16(E[c])) return PIC_ERR_INVALID_ARG;
    if ((in->n > 0 && !aligned16(perm)) || !aligned16(cell_offsets)) return PIC_ERR_INVALID_ARG;
    if (in->n > 0 && aliases(*grid, *in, *out, in->n)) return PIC_ERR_INVALID_ARG;
    if ((rc = field_supported(*grid)) != PIC_OK) return rc;          // before the sort and the deposit are enqueued
    const size_t sb = sort_ws_bytes(*grid, in->n);
    if (ws_bytes < sb + field_ws_bytes(*grid)) return PIC_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    SortWs sws;
    if ((rc = carve_sort_ws(*grid, in->n, ws, sb, sws)) != PIC_OK) return rc;
    pic_particles_t o = *out;
    o.n = in->n;
    if ((rc = launch_sort(*grid, *in, o, perm, cell_offsets, sws, false, false, st)) != PIC_OK) return rc;
    rc = launch_selfconsistent(*grid, *in, o, perm, sws, rho, E, (char*)ws + sb, dt, qm, st);
    mark_phase(PIC_PHASE_PUSH, st);
    return rc;
}

// ---- host-buffer entry point: the end-to-end path bench.py times ---------------------------
struct HostLayout {
    size_t in[7], out[7], perm, offsets, rho, E[3], ws, total, ws_bytes;
};

static HostLayout host_layout(const pic_grid_t& g, int64_t n)
{
    HostLayout L;
    const size_t s = g.dtype == PIC_F64 ? 8 : 4;
    const size_t C = (size_t)cells_of(g);
    const size_t nb = align256(s * (size_t)(n > 0 ? n : 1));
    size_t off = 0;
    for (int a = 0; a < 7; ++a) { L.in[a] = off; off += nb; }
    for (int a = 0; a < 7; ++a) { L.out[a] = off; off += nb; }
    L.perm = off; off += align256(4 * (size_t)(n > 0 ? n : 1));
    L.offsets = off; off += align256(4 * (C + 1));
    L.rho = off; off += align256(s * C);
    for (int c = 0; c < 3; ++c) { L.E[c] = off; off += align256(s * C); }
    L.ws = off;
    L.ws_bytes = sort_ws_bytes(g, n);
    off += L.ws_bytes;
    L.total = off;
    return L;
}

int pic_step_host_bytes(const pic_grid_t* grid, int64_t n, size_t* bytes)
{
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if (!bytes || n < 0 || n >= ((int64_t)1 << 30)) return PIC_ERR_INVALID_ARG;
    *bytes = host_layout(*grid, n).total;
    return PIC_OK;
}

int pic_step_host(const pic_grid_t* grid, const pic_particles_t* in, pic_particles_t* out, int32_t* perm,
                  int32_t* cell_offsets, void* rho, const void* const E[3], double dt, double qm, int do_sort,
                  void* dev_ws, size_t dev_ws_bytes, void* stream)
{
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if (!in || !out || in->n < 0 || in->n >= ((int64_t)1 << 30) || !E || !rho || !aligned16(dev_ws))
        return PIC_ERR_INVALID_ARG;
    if (do_sort && (!perm || !cell_offsets)) return PIC_ERR_INVALID_ARG;
    const pic_grid_t& g = *grid;
    const int64_t n = in->n;
    HostLayout L = host_layout(g, n);
    if (dev_ws_bytes < L.total) return PIC_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    char* b = (char*)dev_ws;
    const size_t s = g.dtype == PIC_F64 ? 8 : 4;
    const size_t C = (size_t)cells_of(g);

    pic_particles_t din, dout;
    memset(&din, 0, sizeof(din));
    memset(&dout, 0, sizeof(dout));
    din.n = dout.n = n;
    const void* dE[3] = {nullptr, nullptr, nullptr};
    for (int c = 0; c < g.dim; ++c) {
        if (!in->x[c] || !in->v[c] || !out->x[c] || !out->v[c] || !E[c]) return PIC_ERR_INVALID_ARG;
        din.x[c] = b + L.in[c];      din.v[c] = b + L.in[3 + c];
        dout.x[c] = b + L.out[c];    dout.v[c] = b + L.out[3 + c];
        dE[c] = b + L.E[c];
    }
    if (!in->w || !out->w) return PIC_ERR_INVALID_ARG;
    din.w = b + L.in[6];
    dout.w = b + L.out[6];
    int32_t* dperm = (int32_t*)(b + L.perm);
    int32_t* doff = (int32_t*)(b + L.offsets);
    void* drho = b + L.rho;

    for (int c = 0; c < g.dim; ++c) {
        PIC_CUDA_OK(cudaMemcpyAsync(din.x[c], in->x[c], s * (size_t)n, cudaMemcpyHostToDevice, st));
        PIC_CUDA_OK(cudaMemcpyAsync(din.v[c], in->v[c], s * (size_t)n, cudaMemcpyHostToDevice, st));
        PIC_CUDA_OK(cudaMemcpyAsync((void*)dE[c], E[c], s * C, cudaMemcpyHostToDevice, st));
    }
    PIC_CUDA_OK(cudaMemcpyAsync(din.w, in->w, s * (size_t)n, cudaMemcpyHostToDevice, st));
    if (!do_sort && cell_offsets)
        PIC_CUDA_OK(cudaMemcpyAsync(doff, cell_offsets, 4 * (C + 1), cudaMemcpyHostToDevice, st));

    rc = pic_step(grid, &din, &dout, dperm, (do_sort || cell_offsets) ? doff : nullptr, drho, dE, dt, qm,
                  do_sort ? PIC_SORT : 0,              // the particles arrive afresh with every call: never a chain
                  b + L.ws, L.ws_bytes, stream);
    if (rc != PIC_OK) return rc;
    const int launches = g_launches;

    for (int c = 0; c < g.dim; ++c) {
        PIC_CUDA_OK(cudaMemcpyAsync(out->x[c], dout.x[c], s * (size_t)n, cudaMemcpyDeviceToHost, st));
        PIC_CUDA_OK(cudaMemcpyAsync(out->v[c], dout.v[c], s * (size_t)n, cudaMemcpyDeviceToHost, st));
    }
    PIC_CUDA_OK(cudaMemcpyAsync(out->w, dout.w, s * (size_t)n, cudaMemcpyDeviceToHost, st));
    PIC_CUDA_OK(cudaMemcpyAsync(rho, drho, s * C, cudaMemcpyDeviceToHost, st));
    if (do_sort) {
        PIC_CUDA_OK(cudaMemcpyAsync(perm, dperm, 4 * (size_t)n, cudaMemcpyDeviceToHost, st));
        PIC_CUDA_OK(cudaMemcpyAsync(cell_offsets, doff, 4 * (C + 1), cudaMemcpyDeviceToHost, st));
    }
    PIC_CUDA_OK(cudaStreamSynchronize(st));
    g_launches = launches;
    return PIC_OK;
}

// ---- particles resident on the device, grid quantities on the host --------------------------
int pic_step_fields_host_bytes(const pic_grid_t* grid, int64_t n, size_t* bytes)
{
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if (!bytes || n < 0 || n >= ((int64_t)1 << 30)) return PIC_ERR_INVALID_ARG;
    const size_t s = grid->dtype == PIC_F64 ? 8 : 4;
    *bytes = 4 * align256(s * (size_t)cells_of(*grid)) + sort_ws_bytes(*grid, n);
    return PIC_OK;
}

int pic_step_fields_host(const pic_grid_t* grid, const pic_particles_t* in, pic_particles_t* out, int32_t* perm,
                         int32_t* cell_offsets, void* rho, const void* const E[3], double dt, double qm, int do_sort,
                         void* ws, size_t ws_bytes, void* stream)
{
    int rc = check_grid(grid);
    if (rc != PIC_OK) return rc;
    if (!rho || !E || !aligned16(ws)) return PIC_ERR_INVALID_ARG;
    const size_t s = grid->dtype == PIC_F64 ? 8 : 4;
    const size_t C = (size_t)cells_of(*grid), gb = align256(s * C);
    const size_t need = 4 * gb + sort_ws_bytes(*grid, in ? in->n : 0);
    if (!in || ws_bytes < need) return in ? PIC_ERR_WORKSPACE : PIC_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    char* b = (char*)ws;
    const void* dE[3] = {nullptr, nullptr, nullptr};
    for (int c = 0; c < grid->dim; ++c) {
        if (!E[c]) return PIC_ERR_INVALID_ARG;
        dE[c] = b + (size_t)c * gb;
        PIC_CUDA_OK(cudaMemcpyAsync(b + (size_t)c * gb, E[c], s * C, cudaMemcpyHostToDevice, st));
    }
    void* drho = b + 3 * gb;
    rc = pic_step(grid, in, out, perm, cell_offsets, drho, dE, dt, qm, do_sort, b + 4 * gb, ws_bytes - 4 * gb, stream);
    if (rc != PIC_OK) return rc;
    const int launches = g_launches;
    PIC_CUDA_OK(cudaMemcpyAsync(rho, drho, s * C, cudaMemcpyDeviceToHost, st));
    PIC_CUDA_OK(cudaStreamSynchronize(st));
    g_launches = launches;
    return PIC_OK;
}

}  // extern "C"
