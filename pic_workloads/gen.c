/*
 * pic_workloads/gen.c -- seeded synthetic inputs shaped like the paper's workload.
 *
 * This module holds NONE of the method's arithmetic (no keys, no splines, no
 * push): it only draws the random numbers and evaluates the prescribed field
 * that both the CPU oracle (oracle/) and the CUDA path are then fed with.
 *
 * Workload shape: "Particles are pseudo-randomly loaded uniformly between the
 * system bounds" on a uniform periodic grid, with a frozen, prescribed E
 * (section 3; section 5).  Recipe: DESIGN.md
 * "Input recipe".
 *
 * RNG: counter based, index addressable.
 *   mix64  = the splitmix64 output function (Steele, Lea, Flood 2014)
 *   key    = mix64(seed + G*(stream+1)),  G = 0x9E3779B97F4A7C15
 *   r(i)   = mix64(key  + G*(i+1))
 *   u(i)   = (r >> 11) * 2^-53   in [0,1)
 * Every element depends only on (seed, stream, index), so the fill loops are
 * OpenMP-parallel without changing a single bit of the output.
 * Normals: Box-Muller in double from two streams (a,b):
 *   z = sqrt(-2 ln(1-u_a)) * cos(2 pi u_b)
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

#define PICW_G 0x9E3779B97F4A7C15ULL

static inline uint64_t mix64(uint64_t z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

static inline uint64_t stream_key(uint64_t seed, uint64_t stream)
{
    return mix64(seed + PICW_G * (stream + 1));
}

static inline double u01(uint64_t key, uint64_t i)
{
    return (double)(mix64(key + PICW_G * (i + 1)) >> 11) * (1.0 / 9007199254740992.0);
}

static inline void store(void *out, int is_f64, int64_t i, double v)
{
    if (is_f64) ((double *)out)[i] = v;
    else        ((float  *)out)[i] = (float)v;
}

/* u(seed,stream,i0..i0+n) as doubles (exposed so tests can cross-check the RNG) */
void picw_uniform01(uint64_t seed, uint64_t stream, int64_t i0, int64_t n, double *out)
{
    uint64_t key = stream_key(seed, stream);
    for (int64_t i = 0; i < n; ++i) out[i] = u01(key, (uint64_t)(i0 + i));
}

/* out[i] = lo + (hi-lo)*u, rounded once to the storage dtype; a value that
 * rounds to >= wrap (when wrap > 0) becomes 0 so that 0 <= x < L holds in storage. */
void picw_fill_uniform(uint64_t seed, uint64_t stream, int64_t n, double lo, double hi,
                       double wrap, int is_f64, void *out)
{
    uint64_t key = stream_key(seed, stream);
    #pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double v = lo + (hi - lo) * u01(key, (uint64_t)i);
        if (wrap > 0.0) {
            double s = is_f64 ? v : (double)(float)v;
            if (s >= wrap || s < 0.0) v = 0.0;
        }
        store(out, is_f64, i, v);
    }
}

/* out[i] = mean + sigma * z_i, z by Box-Muller from streams (sa, sb) */
void picw_fill_normal(uint64_t seed, uint64_t sa, uint64_t sb, int64_t n, double mean,
                      double sigma, int is_f64, void *out)
{
    const double two_pi = 6.283185307179586476925286766559;
    uint64_t ka = stream_key(seed, sa), kb = stream_key(seed, sb);
    #pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double ua = u01(ka, (uint64_t)i), ub = u01(kb, (uint64_t)i);
        double z = sqrt(-2.0 * log(1.0 - ua)) * cos(two_pi * ub);
        store(out, is_f64, i, mean + sigma * z);
    }
}

/* Clustered positions of BASELINE.json config 4: particle i belongs to the blob
 * when u(ssel,i) < frac: x = centre + sigma*z folded into [0,L); else uniform. */
void picw_fill_clustered(uint64_t seed, uint64_t ssel, uint64_t su, uint64_t sa, uint64_t sb,
                         int64_t n, double frac, double centre, double sigma, double L,
                         int is_f64, void *out)
{
    const double two_pi = 6.283185307179586476925286766559;
    uint64_t ksel = stream_key(seed, ssel), ku = stream_key(seed, su);
    uint64_t ka = stream_key(seed, sa), kb = stream_key(seed, sb);
    #pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double v;
        if (u01(ksel, (uint64_t)i) < frac) {
            double ua = u01(ka, (uint64_t)i), ub = u01(kb, (uint64_t)i);
            v = centre + sigma * sqrt(-2.0 * log(1.0 - ua)) * cos(two_pi * ub);
            v -= L * floor(v / L);
        } else {
            v = L * u01(ku, (uint64_t)i);
        }
        double s = is_f64 ? v : (double)(float)v;
        if (s >= L || s < 0.0) v = 0.0;
        store(out, is_f64, i, v);
    }
}

/* Prescribed, frozen electrostatic field from M plane-wave modes, sampled on the
 * nodes j*h of an n[0] x n[1] x n[2] periodic grid (x fastest):
 *   E_c[j] = sum_m amp[m] * dir[m][c] * sin(2 pi sum_c' k[m][c'] j_c'/n_c' + phase[m])
 * k: integer wave vectors [M][3]; dir: unit direction [M][3] (the caller passes
 * k/|k| for an electrostatic field, or any fixed direction). */
void picw_field_modes(int dim, const int32_t *n, int M, const int32_t *k, const double *dir,
                      const double *amp, const double *phase, int comp, int is_f64, void *out)
{
    const double two_pi = 6.283185307179586476925286766559;
    int64_t nx = n[0], ny = n[1], nz = (dim == 3) ? n[2] : 1;
    #pragma omp parallel for collapse(2) schedule(static)
    for (int64_t jz = 0; jz < nz; ++jz)
        for (int64_t jy = 0; jy < ny; ++jy)
            for (int64_t jx = 0; jx < nx; ++jx) {
                double e = 0.0;
                for (int m = 0; m < M; ++m) {
                    double ph = (double)k[3 * m + 0] * (double)jx / (double)nx
                              + (double)k[3 * m + 1] * (double)jy / (double)ny;
                    if (dim == 3) ph += (double)k[3 * m + 2] * (double)jz / (double)nz;
                    e += amp[m] * dir[3 * m + comp] * sin(two_pi * ph + phase[m]);
                }
                store(out, is_f64, jx + nx * (jy + ny * jz), e);
            }
}
