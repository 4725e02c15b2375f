// pic_field.cu -- pic_field_solve: step ii of the loop, "field_solver(): -Laplace(phi) = rho" (section 3;
// "we solve Poisson's equation for computing the field potential phi"), periodic.  The paper
// leaves the step out ("not considered"): SURVEY 8(f) NEXT-4.  Readings R21-R23:
// E = -grad(phi); the mean of rho is dropped and phi has zero mean; spectral discretisation on the node grid,
//     phi^ = rho^ / sum_c kappa_c^2,  E_c^ = -i kappa'_c phi^,  kappa_c(m) = 2 pi mt / L_c (mt = m up to n/2, m - n above),
//     kappa' = kappa except 0 at the Nyquist index of an even n.
//
// The grids are small next to the particles (2^21 nodes on cfg3: 33 MB as complex doubles, resident in L2), so the
// solve is done in double whatever the storage type, one transform axis at a time:
//   k_load_real      rho (T) -> complex double
//   k_fft_axis       all lines of one axis: a block stages a few neighbouring lines in shared memory; power-of-two
//                    lengths run a Stockham radix-2 FFT there (no bit reversal), other lengths the plain DFT sum
//   k_spectral       B = A / kappa^2   or   B = -i kappa'_c A / kappa^2
//   k_store_real     Re(B) / C -> phi or E_c (T)
// Hand-written: no cuFFT.  Twiddles come from sincospi in double.
#include "pic_common.cuh"

namespace pic {

typedef double2 cplx;

__device__ __forceinline__ cplx cmul(cplx a, cplx b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

template <typename T>
__global__ void __launch_bounds__(256) k_load_real(const T* __restrict__ in, cplx* __restrict__ out, int64_t C)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < C) out[k] = make_double2((double)in[k], 0.0);
}

template <typename T>
__global__ void __launch_bounds__(256) k_store_real(const cplx* __restrict__ in, T* __restrict__ out, int64_t C, double scale)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < C) out[k] = (T)(in[k].x * scale);
}

// One axis of length n: element k of line l sits at (l % inner) + (l / inner) * inner * n + k * inner, inner = number of
// nodes below the axis (1 for x).  A block takes LB consecutive lines: for y and z they are neighbours in memory.
// sign = -1 forward, +1 inverse (unscaled).  In place: a block reads its lines completely before it writes them.
template <bool POW2>
__global__ void __launch_bounds__(256) k_fft_axis(cplx* __restrict__ data, int n, int64_t inner, int64_t nlines, int LB, double sign)
{
    extern __shared__ __align__(16) unsigned char s_raw[];
    cplx* tw = reinterpret_cast<cplx*>(s_raw);              // [n] exp(sign 2 pi i k / n)
    cplx* buf0 = tw + n;                                    // [LB][n]
    cplx* buf1 = buf0 + (size_t)LB * n;                     // [LB][n]
    const int tid = threadIdx.x, nt = blockDim.x;
    const int64_t l0 = (int64_t)blockIdx.x * LB;
    const int lines = (int)((nlines - l0 < LB) ? (nlines - l0) : LB);
    for (int k = tid; k < n; k += nt) {
        double s, c;
        sincospi(2.0 * (double)k / (double)n, &s, &c);
        tw[k] = make_double2(c, sign * s);
    }
    const bool lines_fast = inner > 1;                      // consecutive threads on consecutive lines (contiguous in memory)
    for (int idx = tid; idx < lines * n; idx += nt) {
        const int ll = lines_fast ? idx % lines : idx / n, k = lines_fast ? idx / lines : idx % n;
        const int64_t l = l0 + ll;
        buf0[(size_t)ll * n + k] = data[(l % inner) + (l / inner) * inner * n + (int64_t)k * inner];
    }
    __syncthreads();
    cplx* src = buf0;
    cplx* dst = buf1;
    if constexpr (POW2) {
        const int half = n >> 1;
        for (int ncur = n, s = 1; ncur > 1; ncur >>= 1, s <<= 1) {
            const int m = ncur >> 1;
            for (int t = tid; t < lines * half; t += nt) {
                const int ll = t / half, u = t - ll * half;
                const int p = u / s, q = u - p * s;
                const cplx a = src[(size_t)ll * n + q + s * p], b = src[(size_t)ll * n + q + s * (p + m)];
                const cplx w = tw[p * s];
                dst[(size_t)ll * n + q + s * 2 * p] = make_double2(a.x + b.x, a.y + b.y);
                dst[(size_t)ll * n + q + s * (2 * p + 1)] = cmul(make_double2(a.x - b.x, a.y - b.y), w);
            }
            __syncthreads();
            cplx* t2 = src; src = dst; dst = t2;
        }
    } else {
        for (int idx = tid; idx < lines * n; idx += nt) {
            const int ll = idx / n, k = idx - ll * n;
            double re = 0.0, im = 0.0;
            int ph = 0;                                     // (j k) mod n
            for (int j = 0; j < n; ++j) {
                const cplx a = src[(size_t)ll * n + j], w = tw[ph];
                re += a.x * w.x - a.y * w.y;
                im += a.x * w.y + a.y * w.x;
                ph += k;
                if (ph >= n) ph -= n;
            }
            dst[(size_t)ll * n + k] = make_double2(re, im);
        }
        __syncthreads();
        src = dst;
    }
    for (int idx = tid; idx < lines * n; idx += nt) {
        const int ll = lines_fast ? idx % lines : idx / n, k = lines_fast ? idx / lines : idx % n;
        const int64_t l = l0 + ll;
        data[(l % inner) + (l / inner) * inner * n + (int64_t)k * inner] = src[(size_t)ll * n + k];
    }
}

struct SpecP {
    int n[3];
    double two_pi_over_L[3];
};

// comp < 0: B = A / kappa^2 (phi^); else B = -i kappa'_comp A / kappa^2 (E_comp^); the mean (kappa = 0) is dropped
__global__ void __launch_bounds__(256) k_spectral(const cplx* __restrict__ A, cplx* __restrict__ B, SpecP sp, int64_t C, int comp)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= C) return;
    int m[3];
    m[0] = (int)(k % sp.n[0]);
    m[1] = (int)((k / sp.n[0]) % sp.n[1]);
    m[2] = (int)(k / ((int64_t)sp.n[0] * sp.n[1]));
    double k2 = 0.0, kd = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int n = sp.n[c];
        const int mt = (2 * m[c] <= n) ? m[c] : m[c] - n;
        const double kap = sp.two_pi_over_L[c] * (double)mt;
        k2 += kap * kap;
        if (c == comp) kd = (n % 2 == 0 && 2 * m[c] == n) ? 0.0 : kap;
    }
    const cplx a = A[k];
    cplx b = make_double2(0.0, 0.0);
    if (k != 0) {
        const double inv = 1.0 / k2;
        if (comp < 0) b = make_double2(a.x * inv, a.y * inv);
        else b = make_double2(a.y * kd * inv, -a.x * kd * inv);
    }
    B[k] = b;
}

static inline size_t align256f(size_t b) { return (b + 255) & ~(size_t)255; }

size_t field_ws_bytes(const pic_grid_t& g)
{
    size_t C = 1;
    for (int c = 0; c < g.dim; ++c) C *= (size_t)g.n[c];
    return 2 * align256f(sizeof(cplx) * C);
}

// lines per block and dynamic shared memory for an axis of length n (0: too long for this build)
constexpr size_t kFieldSmemBudget = 200 * 1024;
constexpr int kFieldMaxN = 4096;          // the bound pic.h documents (the shared-memory budget alone would allow 4266)
static int lines_per_block(int n, size_t& smem)
{
    const size_t budget = kFieldSmemBudget;
    if (n > kFieldMaxN) { smem = 0; return 0; }
    int lb = 8;
    while (lb > 1 && sizeof(cplx) * ((size_t)2 * lb * n + n) > 64 * 1024) lb >>= 1;
    smem = sizeof(cplx) * ((size_t)2 * lb * n + n);
    return smem <= budget ? lb : 0;
}

// PIC_OK if every axis has a transform in this build, else PIC_ERR_UNSUPPORTED: asked BEFORE anything is enqueued
int field_supported(const pic_grid_t& g)
{
    for (int c = 0; c < g.dim; ++c) {
        size_t smem = 0;
        if (lines_per_block(g.n[c], smem) == 0) return PIC_ERR_UNSUPPORTED;
    }
    return PIC_OK;
}

// The transforms of long axes need more dynamic shared memory than the default limit: raised to the budget once per
// device and kernel, not on every call.
template <bool POW2>
static int raise_smem_limit_once()
{
    static bool done[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return PIC_ERR_CUDA;
    if (dev >= 0 && dev < 64 && done[dev]) return PIC_OK;
    PIC_CUDA_OK(cudaFuncSetAttribute(k_fft_axis<POW2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFieldSmemBudget));
    if (dev >= 0 && dev < 64) done[dev] = true;
    return PIC_OK;
}

static int fft_all_axes(const pic_grid_t& g, cplx* data, double sign, cudaStream_t st)
{
    int64_t C = 1;
    for (int c = 0; c < g.dim; ++c) C *= g.n[c];
    int64_t inner = 1;
    for (int c = 0; c < g.dim; ++c) {
        const int n = g.n[c];
        size_t smem = 0;
        const int lb = lines_per_block(n, smem);
        if (lb == 0) return PIC_ERR_UNSUPPORTED;
        const int64_t nlines = C / n;
        const unsigned blocks = (unsigned)((nlines + lb - 1) / lb);
        const bool pow2 = (n & (n - 1)) == 0;
        auto kern = pow2 ? k_fft_axis<true> : k_fft_axis<false>;
        if (smem > 48 * 1024) {
            const int rc = pow2 ? raise_smem_limit_once<true>() : raise_smem_limit_once<false>();
            if (rc != PIC_OK) return rc;
        }
        kern<<<blocks, 256, smem, st>>>(data, n, inner, nlines, lb, sign);
        count_launch();
        inner *= n;
    }
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

template <typename T>
static int field_impl(const pic_grid_t& g, const void* rho, void* const E[3], void* phi, void* ws, cudaStream_t st)
{
    int64_t C = 1;
    SpecP sp;
    for (int c = 0; c < 3; ++c) {
        sp.n[c] = c < g.dim ? g.n[c] : 1;
        sp.two_pi_over_L[c] = c < g.dim ? 2.0 * 3.14159265358979323846 / ((double)g.n[c] * g.h[c]) : 0.0;
        C *= sp.n[c];
    }
    cplx* A = (cplx*)ws;
    cplx* B = (cplx*)((char*)ws + align256f(sizeof(cplx) * (size_t)C));
    const unsigned blocks = (unsigned)((C + 255) / 256);
    k_load_real<T><<<blocks, 256, 0, st>>>((const T*)rho, A, C);
    count_launch();
    int rc = fft_all_axes(g, A, -1.0, st);
    if (rc != PIC_OK) return rc;
    for (int comp = phi ? -1 : 0; comp < g.dim; ++comp) {
        k_spectral<<<blocks, 256, 0, st>>>(A, B, sp, C, comp);
        count_launch();
        if ((rc = fft_all_axes(g, B, +1.0, st)) != PIC_OK) return rc;
        k_store_real<T><<<blocks, 256, 0, st>>>(B, (T*)(comp < 0 ? phi : E[comp]), C, 1.0 / (double)C);
        count_launch();
    }
    return cudaPeekAtLastError() == cudaSuccess ? PIC_OK : PIC_ERR_CUDA;
}

int launch_field_solve(const pic_grid_t& g, const void* rho, void* const E[3], void* phi, void* ws, cudaStream_t st)
{
    return g.dtype == PIC_F32 ? field_impl<float>(g, rho, E, phi, ws, st) : field_impl<double>(g, rho, E, phi, ws, st);
}

}  // namespace pic
