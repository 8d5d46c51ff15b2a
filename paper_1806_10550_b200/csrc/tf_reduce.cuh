// tf_reduce.cuh -- reductions of a field (S9 mass of (3.2), and the validity check of a state).
#pragma once
#include "tf_device.cuh"

namespace tf {

constexpr int XT = 32;          // tile edge of the transposing kernels (tf_penta.cuh)
constexpr int XTP = XT + 1;     // padded row length (doubles)
constexpr int PF = 8;           // rows of register prefetch in the simple marching kernels

// ---------------------------------------------------------------------------------------------
// reductions (S9 mass, state validation): fixed grid, fixed order -> bitwise reproducible
// ---------------------------------------------------------------------------------------------
constexpr int RED_BLOCKS = 1184;   // 8 x 148 SMs
constexpr int RED_THREADS = 256;

// part[b] = sum over a fixed slice; flag[0] |= any non-finite or non-positive value
__global__ void __launch_bounds__(RED_THREADS)
sum_check_kernel(size_t n, const double* __restrict__ h, double* __restrict__ part, int* __restrict__ flag)
{
    __shared__ double sm[RED_THREADS / 32];
    double acc = 0.0;
    int bad = 0;
    for (size_t p = (size_t)blockIdx.x * RED_THREADS + threadIdx.x; p < n; p += (size_t)RED_BLOCKS * RED_THREADS) {
        const double v = h[p];
        acc += v;
        if (!(v > 0.0) || isinf(v)) bad = 1;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = acc;
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(flag, 1);
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < RED_THREADS / 32; ++k) t += sm[k];
        part[blockIdx.x] = t;
    }
}

// extra solution criterion of Fig. 1 (PAPER.md:252 Note 2): out[0] = max |u_new - u_old| / u_old over the field
// (order-independent max on the bit patterns of non-negative doubles -> bitwise reproducible; NaN surfaces)
__device__ __forceinline__ void
max_rel_change_body(size_t n, const double* __restrict__ u_old, const double* __restrict__ u_new, double* __restrict__ out)
{
    double acc = 0.0;
    for (size_t p = (size_t)blockIdx.x * RED_THREADS + threadIdx.x; p < n; p += (size_t)RED_BLOCKS * RED_THREADS) {
        const double o = u_old[p];
        const double r = fabs(u_new[p] - o) / o;
        acc = (r != r) ? __longlong_as_double(0x7ff8000000000000LL) : ((acc != acc) ? acc : fmax(acc, r));
    }
    acc = warp_max_nonneg(acc);
    if ((threadIdx.x & 31) == 0) atomic_max_nonneg(out, acc);
}

// Truncation-error estimate of the trapezoidal rule (PAPER.md:252 Note 2 "sufficiently small truncation error"; reading
// R25 of DESIGN.md): the local error of (2.14) is -(dt^3/12) u_ttt.  With u_t^n = -D(u^n) = 2 (b^n - u^n)/dt and the
// Crank-Nicolson relation u_t^{n+1} = 2 (u^{n+1} - u^n)/dt - u_t^n, the second time derivative at the midpoint of the step is
//   a_{n+1/2} = (u_t^{n+1} - u_t^n)/dt = 2 (u^{n+1} + u^n - 2 b^n)/dt^2,
// and u_ttt ~ (a_{n+1/2} - a_{n-1/2}) / ((dt + dt_prev)/2) with a_{n-1/2} kept from the previous accepted step.
// Writes a_{n+1/2} to a_new (committed by the host only if the step is accepted) and max |tau| / |u^{n+1}| to out.
// have_prev == 0 (first step after tf_set_state): only a_new is written.
__global__ void __launch_bounds__(RED_THREADS)
max_rel_change_kernel(size_t n, const double* __restrict__ u_old, const double* __restrict__ u_new, double* __restrict__ out)
{
    max_rel_change_body(n, u_old, u_new, out);
}

__device__ __forceinline__ void
truncation_body(size_t n, const double* __restrict__ u_old, const double* __restrict__ u_new, const double* __restrict__ bn,
                const double* __restrict__ a_prev, double* __restrict__ a_new, double two_over_dt2, double scale,
                int have_prev, double* __restrict__ out)
{
    double acc = 0.0;
    for (size_t p = (size_t)blockIdx.x * RED_THREADS + threadIdx.x; p < n; p += (size_t)RED_BLOCKS * RED_THREADS) {
        const double un = u_new[p];
        const double a = two_over_dt2 * ((un + u_old[p]) - 2.0 * bn[p]);
        a_new[p] = a;
        if (have_prev) {
            const double r = scale * fabs(a - a_prev[p]) / fabs(un);     // scale = (dt^3/12) / ((dt + dt_prev)/2)
            acc = (r != r) ? __longlong_as_double(0x7ff8000000000000LL) : ((acc != acc) ? acc : fmax(acc, r));
        }
    }
    acc = warp_max_nonneg(acc);
    if ((threadIdx.x & 31) == 0) atomic_max_nonneg(out, acc);
}

__global__ void __launch_bounds__(RED_THREADS)
truncation_kernel(size_t n, const double* __restrict__ u_old, const double* __restrict__ u_new, const double* __restrict__ bn,
                  const double* __restrict__ a_prev, double* __restrict__ a_new, double two_over_dt2, double scale,
                  int have_prev, double* __restrict__ out)
{
    truncation_body(n, u_old, u_new, bn, a_prev, a_new, two_over_dt2, scale, have_prev, out);
}

// The same two reductions for the on-device controller (tf_control.cuh): they run only if the attempt converged
// (`conv`), and the truncation estimate takes dt, dt_prev and "a history exists" from device memory.  The scalars are
// formed by the operations tf_step uses on the host, in its order, none of them contractible into an FMA: same bits.
__global__ void __launch_bounds__(RED_THREADS)
max_rel_change_ctl_kernel(size_t n, const double* __restrict__ u_old, const double* __restrict__ u_new,
                          const double* __restrict__ conv, double* __restrict__ out)
{
    if (__ldcg(conv) == 0.0) return;
    max_rel_change_body(n, u_old, u_new, out);
}

__global__ void __launch_bounds__(RED_THREADS)
truncation_ctl_kernel(size_t n, const double* __restrict__ u_old, const double* __restrict__ u_new, const double* __restrict__ bn,
                      const double* __restrict__ a_prev, double* __restrict__ a_new, const double* __restrict__ conv,
                      const double* __restrict__ dt_p, const double* __restrict__ dt_prev_p, const double* __restrict__ have_p,
                      double* __restrict__ out)
{
    if (__ldcg(conv) == 0.0) return;
    const double dt = __ldcg(dt_p), dt_prev = __ldcg(dt_prev_p);
    const int have = __ldcg(have_p) != 0.0 ? 1 : 0;
    const double dt2 = __dmul_rn(dt, dt);
    const double scale = have ? __ddiv_rn(__ddiv_rn(__dmul_rn(dt2, dt), 12.0), __dmul_rn(0.5, __dadd_rn(dt, dt_prev))) : 0.0;
    truncation_body(n, u_old, u_new, bn, a_prev, a_new, __ddiv_rn(2.0, dt2), scale, have, out);
}

__global__ void __launch_bounds__(1024)
sum_final_kernel(const double* __restrict__ part, double scale, double* __restrict__ out)
{
    __shared__ double sm[1024];
    const int t = threadIdx.x;
    sm[t] = (t < RED_BLOCKS ? part[t] : 0.0) + (t + 1024 < RED_BLOCKS ? part[t + 1024] : 0.0);
    __syncthreads();
    for (int o = 512; o > 0; o >>= 1) {
        if (t < o) sm[t] += sm[t + o];
        __syncthreads();
    }
    if (t == 0) out[0] = scale * sm[0];
}

}  // namespace tf
