// pic_stencil.cuh -- pieces shared by the kernels that work on particles grouped by cell
// (pic_runs.cuh, pic_tile.cuh, pic_nodes.cu) and by the any-order kernels: field pointers, kernel modes, the
// stencil width of a cell, packed pairs, the 1-D spline weights of a cell's stencil.
//
// S = stencil width of a CELL: 2 for p = 1, 4 for p = 2, 3 (a quadratic particle touches 3 of the
// 4 nodes i0-1..i0+2, which 3 depends on xi >= 1/2; the fourth weight is an exact zero).
// Arithmetic on pairs of x-neighbouring nodes uses the packed fp32 instructions of sm_100
// (fma.rn.f32x2, SASS FFMA2): half the issue slots of two scalar FMAs.
#pragma once
#include "pic_common.cuh"

namespace pic {

template <typename T>
struct FieldP {
    const T* E[3];
};

enum { kModeDeposit = 1, kModePush = 2, kModeBoth = 3 };

template <int P>
struct StencilW {
    static constexpr int S = (P == 1) ? 2 : 4;
};

// ---------------------------------------------------------------------------------------------
// packed pairs: fp32 pairs live in one 64-bit register and use the f32x2 instructions
template <typename T>
struct Pk;
template <>
struct Pk<float> {
    unsigned long long r;
};
template <>
struct Pk<double> {
    double lo, hi;
};

__device__ __forceinline__ Pk<float> pk_make(float lo, float hi)
{
    Pk<float> p;
    asm("mov.b64 %0, {%1, %2};" : "=l"(p.r) : "f"(lo), "f"(hi));
    return p;
}
__device__ __forceinline__ Pk<double> pk_make(double lo, double hi) { return Pk<double>{lo, hi}; }
// a pair whose halves the compiler must treat as unrelated (no scalar-broadcast operand form)
__device__ __forceinline__ Pk<float> pk_pair(float lo, float hi)
{
    Pk<float> p;
    asm volatile("mov.b64 %0, {%1, %2};" : "=l"(p.r) : "f"(lo), "f"(hi));
    return p;
}
__device__ __forceinline__ Pk<double> pk_pair(double lo, double hi) { return Pk<double>{lo, hi}; }
__device__ __forceinline__ float pk_lo(Pk<float> p)
{
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p.r));
    (void)hi;
    return lo;
}
__device__ __forceinline__ float pk_hi(Pk<float> p)
{
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p.r));
    (void)lo;
    return hi;
}
__device__ __forceinline__ double pk_lo(Pk<double> p) { return p.lo; }
__device__ __forceinline__ double pk_hi(Pk<double> p) { return p.hi; }
__device__ __forceinline__ Pk<float> pk_fma(Pk<float> a, Pk<float> b, Pk<float> c)
{
    Pk<float> d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d.r) : "l"(a.r), "l"(b.r), "l"(c.r));
    return d;
}
__device__ __forceinline__ Pk<double> pk_fma(Pk<double> a, Pk<double> b, Pk<double> c)
{
    return Pk<double>{fma(a.lo, b.lo, c.lo), fma(a.hi, b.hi, c.hi)};
}
// c += a * b in place (the accumulator is one read-write operand: no copy of a loop-carried sum)
__device__ __forceinline__ void pk_acc(Pk<float>& c, Pk<float> a, Pk<float> b)
{
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(c.r) : "l"(a.r), "l"(b.r));
}
__device__ __forceinline__ void pk_acc(Pk<double>& c, Pk<double> a, Pk<double> b)
{
    c.lo = fma(a.lo, b.lo, c.lo);
    c.hi = fma(a.hi, b.hi, c.hi);
}
__device__ __forceinline__ Pk<float> pk_mul(Pk<float> a, Pk<float> b)
{
    Pk<float> d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d.r) : "l"(a.r), "l"(b.r));
    return d;
}
__device__ __forceinline__ Pk<double> pk_mul(Pk<double> a, Pk<double> b) { return Pk<double>{a.lo * b.lo, a.hi * b.hi}; }
template <typename T>
__device__ __forceinline__ Pk<T> pk_zero()
{
    return pk_make((T)0, (T)0);
}

// weights of one particle on the S-wide stencil of its cell; returns the (clamped) cell index
template <typename T, int P>
__device__ __forceinline__ int cell_weights(T x, T h, T inv_h, int hmul, int n, T (&w)[StencilW<P>::S])
{
    const T t = grid_coord(x, h, inv_h, hmul);
    const int i0 = cell_index(t, n);
    const T xi = t - (T)i0;
    if constexpr (P == 1) {
        w[0] = (T)1 - xi;
        w[1] = xi;
    } else if constexpr (P == 2) {
        const bool up = xi >= (T)0.5;
        const T d = xi - (up ? (T)1 : (T)0);
        const T a = (T)0.5 - d, b = (T)0.5 + d;
        const T w0 = (T)0.5 * a * a, w1 = (T)0.75 - d * d, w2 = (T)0.5 * b * b;
        w[0] = up ? (T)0 : w0;
        w[1] = up ? w0 : w1;
        w[2] = up ? w1 : w2;
        w[3] = up ? w2 : (T)0;
    } else {
        const T om = (T)1 - xi, x2 = xi * xi;
        w[0] = om * om * om * (T)(1.0 / 6.0);
        w[1] = (T)(2.0 / 3.0) - x2 + (T)0.5 * x2 * xi;
        w[2] = (T)(1.0 / 6.0) + (T)0.5 * (xi + x2 - x2 * xi);
        w[3] = x2 * xi * (T)(1.0 / 6.0);
    }
    return i0;
}

// S consecutive values from shared memory as S/2 pairs (128-bit loads)
template <typename T, int S>
__device__ __forceinline__ void load_row(const T* __restrict__ p, Pk<T> (&e)[S / 2])
{
    if constexpr (sizeof(T) == 4 && S == 4) {
        const float4 v = *reinterpret_cast<const float4*>(p);
        e[0] = pk_make(v.x, v.y);
        e[1] = pk_make(v.z, v.w);
    } else if constexpr (sizeof(T) == 4) {
        const float2 v = *reinterpret_cast<const float2*>(p);
        e[0] = pk_make(v.x, v.y);
    } else {
#pragma unroll
        for (int i = 0; i < S / 2; ++i) {
            const double2 v = *reinterpret_cast<const double2*>(p + 2 * i);
            e[i] = pk_make(v.x, v.y);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// shared memory by 32-bit shared-window address.  The base is taken once with a volatile asm, so it
// stays in a register (the compiler otherwise re-derives it from SR_CgaCtaId at every use).
__device__ __forceinline__ uint32_t smem_base(const void* p)
{
    uint32_t a;
    asm volatile("{ .reg .u64 t; cvta.to.shared.u64 t, %1; cvt.u32.u64 %0, t; }" : "=r"(a) : "l"(p));
    return a;
}
// N consecutive elements of T at byte address a (aligned to min(16, N*sizeof(T)))
template <typename T, int N>
__device__ __forceinline__ void lds(uint32_t a, T (&o)[N])
{
    if constexpr (sizeof(T) == 4 && N % 4 == 0) {
#pragma unroll
        for (int i = 0; i < N / 4; ++i)
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                         : "=f"(o[4 * i]), "=f"(o[4 * i + 1]), "=f"(o[4 * i + 2]), "=f"(o[4 * i + 3]) : "r"(a + 16 * i));
    } else if constexpr (sizeof(T) == 4 && N % 2 == 0) {
#pragma unroll
        for (int i = 0; i < N / 2; ++i)
            asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(o[2 * i]), "=f"(o[2 * i + 1]) : "r"(a + 8 * i));
    } else if constexpr (sizeof(T) == 4) {
#pragma unroll
        for (int i = 0; i < N; ++i) asm volatile("ld.shared.f32 %0, [%1];" : "=f"(o[i]) : "r"(a + 4 * i));
    } else if constexpr (N % 2 == 0) {
#pragma unroll
        for (int i = 0; i < N / 2; ++i)
            asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(o[2 * i]), "=d"(o[2 * i + 1]) : "r"(a + 16 * i));
    } else {
#pragma unroll
        for (int i = 0; i < N; ++i) asm volatile("ld.shared.f64 %0, [%1];" : "=d"(o[i]) : "r"(a + 8 * i));
    }
}
// S consecutive elements at byte address a (aligned to 16) as S/2 packed pairs: the fp32 pairs arrive in
// 64-bit registers, so no move packs them
template <int S2>
__device__ __forceinline__ void lds_pairs(uint32_t a, Pk<float> (&o)[S2])
{
    if constexpr (S2 == 2) {
        asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(o[0].r), "=l"(o[1].r) : "r"(a));
    } else {
#pragma unroll
        for (int i = 0; i < S2; ++i) asm volatile("ld.shared.b64 %0, [%1];" : "=l"(o[i].r) : "r"(a + 8 * i));
    }
}
template <int S2>
__device__ __forceinline__ void lds_pairs(uint32_t a, Pk<double> (&o)[S2])
{
#pragma unroll
    for (int i = 0; i < S2; ++i)
        asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(o[i].lo), "=d"(o[i].hi) : "r"(a + 16 * i));
}
template <typename T>
__device__ __forceinline__ T lds1(uint32_t a)
{
    T v[1];
    lds<T, 1>(a, v);
    return v[0];
}
template <typename T, int N>
__device__ __forceinline__ void sts(uint32_t a, const T (&o)[N])
{
    if constexpr (sizeof(T) == 4 && N % 4 == 0) {
#pragma unroll
        for (int i = 0; i < N / 4; ++i)
            asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};"
                         :: "r"(a + 16 * i), "f"(o[4 * i]), "f"(o[4 * i + 1]), "f"(o[4 * i + 2]), "f"(o[4 * i + 3]) : "memory");
    } else if constexpr (sizeof(T) == 4 && N % 2 == 0) {
#pragma unroll
        for (int i = 0; i < N / 2; ++i)
            asm volatile("st.shared.v2.f32 [%0], {%1, %2};" :: "r"(a + 8 * i), "f"(o[2 * i]), "f"(o[2 * i + 1]) : "memory");
    } else if constexpr (sizeof(T) == 4) {
#pragma unroll
        for (int i = 0; i < N; ++i) asm volatile("st.shared.f32 [%0], %1;" :: "r"(a + 4 * i), "f"(o[i]) : "memory");
    } else if constexpr (N % 2 == 0) {
#pragma unroll
        for (int i = 0; i < N / 2; ++i)
            asm volatile("st.shared.v2.f64 [%0], {%1, %2};" :: "r"(a + 16 * i), "d"(o[2 * i]), "d"(o[2 * i + 1]) : "memory");
    } else {
#pragma unroll
        for (int i = 0; i < N; ++i) asm volatile("st.shared.f64 [%0], %1;" :: "r"(a + 8 * i), "d"(o[i]) : "memory");
    }
}
template <typename T>
__device__ __forceinline__ void sts1(uint32_t a, T v)
{
    const T o[1] = {v};
    sts<T, 1>(a, o);
}

// read-only global load that stays where it is written (the compiler may not hoist it: a load issued long
// before its use keeps a scoreboard busy across loop back edges)
__device__ __forceinline__ float ldg_here(const float* p)
{
    float v;
    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ double ldg_here(const double* p)
{
    double v;
    asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}

// asynchronous copy of one element global -> shared (LDGSTS): no register, no scoreboard; wait with cp_async_wait()
__device__ __forceinline__ void cp_async_elem(uint32_t dst, const float* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" :: "r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_elem(uint32_t dst, const double* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// rho[k] = (T) racc[k]
template <typename T>
__global__ void __launch_bounds__(256) k_round_rho(const double* __restrict__ racc, T* __restrict__ rho, int64_t C)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < C) rho[k] = (T)racc[k];
}

}  // namespace pic
