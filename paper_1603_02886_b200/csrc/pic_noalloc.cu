// pic_noalloc.cu -- pic_deposit_static: the fp32 charge deposit for callers that cannot allocate device memory.
//
// Who this is for.  pic_deposit on an fp32 grid adds the particles' contributions into a DOUBLE copy of the grid
// and rounds it into rho once at the end; that double grid is scratch, and pic_deposit takes it from a workspace the
// caller has to allocate (pic_workspace_bytes).  Some callers cannot do that:
//   - a plug-in inside a host application that owns the device heap and hands plug-ins only their input and output
//     buffers (no allocator handle, and a cudaMalloc from the plug-in would break the host's memory accounting);
//   - code that runs between the host application's own kernels on a latency budget, where cudaMalloc/cudaFree are
//     out because both may synchronise the whole device;
//   - a process that starts when the GPU's memory is already handed out to memory pools, so that a late cudaMalloc
//     of a few MiB can fail although the buffers the caller was given are there.
// For them the double grid lives INSIDE THE LIBRARY: a file-scope __device__ array of fixed size, part of the
// library's image on every GPU that loads it (PIC_DEPOSIT_STATIC_MAX_NODES doubles = 16 MiB per GPU, held until the
// process exits).  The caller passes the particles and rho, nothing else.
//
// What is computed: exactly pic_deposit(PIC_ORDER_UNSORTED) -- the paper's "threads on particles" deposit, one
// thread per particle and (p+1)^d atomic additions (setrho 3.3.4), valid for ANY particle order --
// then rho[k] = (float) sum[k].  Same arithmetic per particle as k_deposit_particles in pic_deposit.cu; the two
// differ only in where the double sums live.  The atomics' order is not fixed, so two runs agree to rounding of the
// double sums (about 1e-16 relative, invisible after the rounding to float except for last-bit ties).
//
// The host-side name of a __device__ array is not a device pointer.  Here the name g_racc_static is only a handle
// the runtime looks up: handing `g_racc_static` itself to a kernel from host code would pass a host address (a fault,
// or on a system where the GPU can read host memory a silent write to the wrong place).  The address a kernel
// may use comes from cudaGetSymbolAddress, once per device and with that device current, because every GPU holds
// its own copy of the array at its own address.  static_scratch() below does that and caches the result.
#include <mutex>

#include "pic_common.cuh"

namespace pic {

// 2^21 nodes = a 128^3 grid (the largest grid of BASELINE.json's configs) = 16 MiB of doubles per GPU.
static_assert(PIC_DEPOSIT_STATIC_MAX_NODES == (1 << 21), "pic.h and pic_noalloc.cu disagree about the scratch size");
static __device__ __align__(256) double g_racc_static[PIC_DEPOSIT_STATIC_MAX_NODES];

constexpr int kMaxDevices = 64;
static std::mutex g_scratch_mutex;
static double* g_scratch_ptr[kMaxDevices];      // device address of g_racc_static on device d, or NULL = not looked up yet

// Device address of the CURRENT device's copy of g_racc_static.  The first call on a device asks the runtime
// (cudaGetSymbolAddress; this may load the module onto that device, so it belongs before any stream capture);
// later calls read the cached pointer.  No allocation either way.
static int static_scratch(double** out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return PIC_ERR_CUDA;
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_ptr[dev]) {
        double* ptr = nullptr;
        if (cudaGetSymbolAddress((void**)&ptr, g_racc_static) != cudaSuccess || !ptr) return PIC_ERR_CUDA;
        g_scratch_ptr[dev] = ptr;
    }
    *out = g_scratch_ptr[dev];
    return PIC_OK;
}

// One thread per particle: 1-D spline weights per dimension, then (p+1)^d atomic additions of the products into the
// double grid `racc` (the static array, passed in by address).  Any particle order.
template <int D, int P>
__global__ void __launch_bounds__(256) k_deposit_particles_static(PartP<float> p, GridP<float> g, int64_t n,
                                                                  double* __restrict__ racc)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int first[3] = {0, 0, 0};
    float wt[3][P + 1];
#pragma unroll
    for (int c = 0; c < D; ++c) {
        const float t = grid_coord(p.x[c][i], g.h[c], g.inv_h[c], g.hmul);
        spline_weights<float, P>(t, cell_index(t, g.n[c]), first[c], wt[c]);
    }
    const float q = p.w[i] * g.inv_vol;
#pragma unroll
    for (int cz = 0; cz <= (D == 3 ? P : 0); ++cz) {
        const int jz = D == 3 ? fold(first[2] + cz, g.n[2]) : 0;
        const float qz = D == 3 ? q * wt[2][cz] : q;
#pragma unroll
        for (int b = 0; b <= P; ++b) {
            const int jy = fold(first[1] + b, g.n[1]);
            const float qy = qz * wt[1][b];
            const int64_t row = (int64_t)g.n[0] * (jy + (int64_t)g.n[1] * jz);
#pragma unroll
            for (int a = 0; a <= P; ++a)
                atomicAdd(&racc[row + fold(first[0] + a, g.n[0])], (double)(qy * wt[0][a]));
        }
    }
}

// rho[k] = (float) racc[k]: the one rounding of the fp32 deposit
__global__ void __launch_bounds__(256) k_round_rho_static(const double* __restrict__ racc, float* __restrict__ rho, int64_t C)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < C) rho[k] = (float)racc[k];
}

template <int D, int P>
static void launch_particles_static(const pic_grid_t& g, const pic_particles_t& p, double* racc, cudaStream_t st)
{
    k_deposit_particles_static<D, P><<<(unsigned)((p.n + 255) / 256), 256, 0, st>>>(make_partp<float>(p), make_gridp<float>(g),
                                                                                    p.n, racc);
}

static bool ok16(const void* q) { return q != nullptr && ((uintptr_t)q & 15u) == 0; }

}  // namespace pic

using namespace pic;

extern "C" int pic_deposit_static(const pic_grid_t* grid, const pic_particles_t* p, void* rho, void* stream)
{
    count_launch(-pic_last_launch_count());           // this call's launches only, like every other entry point
    // the same argument rules as pic_deposit, checked before anything is enqueued
    if (!grid || !p) return PIC_ERR_INVALID_ARG;
    if (grid->dim != 2 && grid->dim != 3) return PIC_ERR_INVALID_ARG;
    if (grid->order < 1 || grid->order > 3) return PIC_ERR_INVALID_ARG;
    if (grid->dtype == PIC_F64) return PIC_ERR_UNSUPPORTED;     // fp64 needs no scratch: pic_deposit(ws = NULL) already allocates nothing
    if (grid->dtype != PIC_F32) return PIC_ERR_INVALID_ARG;
    int64_t C = 1;
    for (int c = 0; c < grid->dim; ++c) {
        if (grid->n[c] < grid->order + 1) return PIC_ERR_INVALID_ARG;
        if (!(grid->h[c] > 0.0) || !(grid->h[c] < 1e300)) return PIC_ERR_INVALID_ARG;
        C *= grid->n[c];
        if (C >= ((int64_t)1 << 31)) return PIC_ERR_INVALID_ARG;
    }
    if (C > PIC_DEPOSIT_STATIC_MAX_NODES) return PIC_ERR_TOO_LARGE;
    if (p->n < 0 || p->n >= ((int64_t)1 << 30)) return PIC_ERR_INVALID_ARG;
    if (p->n > 0) {
        for (int c = 0; c < grid->dim; ++c)
            if (!ok16(p->x[c])) return PIC_ERR_INVALID_ARG;
        if (!ok16(p->w)) return PIC_ERR_INVALID_ARG;
    }
    if (!ok16(rho)) return PIC_ERR_INVALID_ARG;

    double* racc = nullptr;
    int rc = static_scratch(&racc);
    if (rc != PIC_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    // the array keeps whatever the last call (of any thread, on any stream) left in it: the sums start from zero
    PIC_CUDA_OK(cudaMemsetAsync(racc, 0, sizeof(double) * (size_t)C, st));
    if (p->n > 0) {
        const int o = grid->order;
        if (grid->dim == 2) {
            if (o == 1) launch_particles_static<2, 1>(*grid, *p, racc, st);
            else if (o == 2) launch_particles_static<2, 2>(*grid, *p, racc, st);
            else launch_particles_static<2, 3>(*grid, *p, racc, st);
        } else {
            if (o == 1) launch_particles_static<3, 1>(*grid, *p, racc, st);
            else if (o == 2) launch_particles_static<3, 2>(*grid, *p, racc, st);
            else launch_particles_static<3, 3>(*grid, *p, racc, st);
        }
        count_launch();
    }
    k_round_rho_static<<<(unsigned)((C + 255) / 256), 256, 0, st>>>(racc, (float*)rho, C);
    count_launch();
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}
