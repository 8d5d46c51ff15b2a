// tf_control.cuh -- the adaptive time-step controller of Fig. 1 taken ON THE DEVICE.
//
// The paper's controller runs on the host and reads a flag array after every iteration.
// Here a whole run of attempts is enqueued without a host round trip: per attempt
//   ctl_begin   (1 CTA)   : opens or closes the attempt (done / enough accepted steps), publishes s = dt/2, clears records
//   K x 4 sweep kernels   : iteration k is gated on iteration k-1's record, iteration 0 on the attempt's gate record;
//                           the forward kernels read s from device memory (Gate::s)
//   ctl_mid     (1 thread): reads the records in order -- the decision of S8 -- and says whether the iteration converged
//   criteria kernels      : only with an extra solution criterion switched on (PAPER.md:252 Note 2): the largest relative
//                           change of h and / or the truncation-error estimate (R25) of a converged attempt, reduced into
//                           the control block; dt, dt_prev and "is there a history" are read from the control block
//   ctl_end     (1 thread): the decision of Fig. 1 -- converged, criteria met -- then accept / shrink / grow exactly as
//                           tf_step + tf_adaptive_run do on the host (same operations in the same order: same status and
//                           dt sequence, bit for bit)
//   ctl_commit  (grid)    : u <- u_(k+1) if the attempt was accepted, a_{n-1/2} <- a_{n+1/2} if the truncation criterion
//                           accepted it (the host path swaps pointers instead)
// The host reads the control block and the attempt history once per enqueued chunk.
#pragma once
#include <cuda_runtime.h>

namespace tf {

// control block, doubles: the layout the host reads back
enum { CT_DT = 0, CT_S, CT_T, CT_ACCEPTED, CT_STREAK, CT_DONE, CT_GATE_RES, CT_GATE_BAD, CT_ATTEMPTS, CT_COMMIT,
       CT_CONV,                  // this attempt's iteration converged (set by ctl_mid; gates the criteria kernels)
       CT_CHANGE, CT_TRUNC,      // criteria of this attempt: max |u_new - u|/u, truncation estimate (max-reduced bit patterns)
       CT_HAVE_ACC, CT_DT_PREV,  // truncation criterion: a_{n-1/2} of the last accepted step is stored / its dt
       CT_COMMIT_ACC,            // this attempt's a_{n+1/2} becomes the stored one
       CT_SIZE = 16 };
constexpr int CT_HIST_CAP = 1024;        // ring of attempt records {dt, status, iters, res}; the host drains it every <= CT_HIST_CAP - 16 attempts
// CT_DONE: 0 running, 1 n_accept reached, 2 dt fell below dt_min, 3 attempt cap reached

struct CtlParams {
    double shrink, grow, dt_min, dt_max, tol;
    double max_rel_change, max_trunc;        // extra solution criteria, 0 = off
    int grow_after, n_accept, max_attempts, kmax;
};

// the decision of S8 from the residual records of one attempt: status 0 (converged) / 1, iteration count, last residual
__device__ __forceinline__ int ctl_scan_records(const double* red, const CtlParams& P, int& k, double& res)
{
    int status = 1;                                       // TF_NOT_CONVERGED
    k = 0; res = 0.0;
    for (int it = 0; it < P.kmax; ++it) {
        k = it + 1;
        res = red[2 * it];
        const bool bad = red[2 * it + 1] != 0.0;
        if (bad || res != res) break;
        if (res < P.tol) { status = 0; break; }
    }
    return status;
}

__global__ void ctl_begin_kernel(double* ctl, double* red, CtlParams P)
{
    for (int k = threadIdx.x; k < 2 * P.kmax; k += blockDim.x) red[k] = 0.0;
    if (threadIdx.x == 0) {
        if (ctl[CT_DONE] == 0.0 && ctl[CT_ACCEPTED] >= (double)P.n_accept) ctl[CT_DONE] = 1.0;
        if (ctl[CT_DONE] == 0.0 && ctl[CT_ATTEMPTS] >= (double)P.max_attempts) ctl[CT_DONE] = 3.0;
        ctl[CT_S] = 0.5 * ctl[CT_DT];
        ctl[CT_GATE_RES] = __longlong_as_double(0x7ff0000000000000LL);   // +inf >= tol: open unless "bad"
        ctl[CT_GATE_BAD] = ctl[CT_DONE] != 0.0 ? 1.0 : 0.0;
        ctl[CT_COMMIT] = 0.0;
        ctl[CT_COMMIT_ACC] = 0.0;
        ctl[CT_CONV] = 0.0;
    }
}

__global__ void ctl_mid_kernel(double* ctl, const double* red, CtlParams P)
{
    if (ctl[CT_GATE_BAD] != 0.0) { ctl[CT_CONV] = 0.0; return; }      // the attempt never ran (the last values stay)
    ctl[CT_CHANGE] = 0.0;
    ctl[CT_TRUNC] = 0.0;
    int k; double res;
    ctl[CT_CONV] = ctl_scan_records(red, P, k, res) == 0 ? 1.0 : 0.0;
}

__global__ void ctl_end_kernel(double* ctl, const double* red, double* hist, CtlParams P)
{
    if (ctl[CT_GATE_BAD] != 0.0) return;                  // the attempt never ran
    int k; double res;
    int status = ctl_scan_records(red, P, k, res);
    const double dt = ctl[CT_DT];
    // the extra solution criteria, in tf_step's order: a converged step is TF_REJECTED (2) if the largest relative change
    // exceeds its limit; if it passes, the truncation estimate is tested (only when a history exists) and, unless that
    // rejects the step, a_{n+1/2} becomes the stored second derivative
    if (status == 0 && P.max_rel_change > 0.0 && !(ctl[CT_CHANGE] <= P.max_rel_change)) status = 2;
    bool commit_acc = false;
    if (status == 0 && P.max_trunc > 0.0) {
        if (ctl[CT_HAVE_ACC] != 0.0 && !(ctl[CT_TRUNC] <= P.max_trunc)) status = 2;
        else commit_acc = true;
    }
    if (status == 0) {
        if (commit_acc) { ctl[CT_COMMIT_ACC] = 1.0; ctl[CT_DT_PREV] = dt; ctl[CT_HAVE_ACC] = 1.0; }
        else ctl[CT_HAVE_ACC] = 0.0;                      // a step taken with the criterion off breaks the history
    }
    const int a = (int)ctl[CT_ATTEMPTS];
    { double* h = hist + 4 * (a % CT_HIST_CAP); h[0] = dt; h[1] = (double)status; h[2] = (double)k; h[3] = res; }   // a ring: the host drains it before it wraps
    ctl[CT_ATTEMPTS] = (double)(a + 1);
    if (status == 0) {
        ctl[CT_ACCEPTED] += 1.0;
        ctl[CT_T] += dt;
        ctl[CT_COMMIT] = 1.0;
        const double streak = ctl[CT_STREAK] + 1.0;
        if (streak >= (double)P.grow_after) { ctl[CT_DT] = fmin(dt * P.grow, P.dt_max); ctl[CT_STREAK] = 0.0; }
        else ctl[CT_STREAK] = streak;
    } else {
        ctl[CT_STREAK] = 0.0;
        const double nd = dt * P.shrink;
        ctl[CT_DT] = nd;
        if (nd < P.dt_min) ctl[CT_DONE] = 2.0;
    }
}

__global__ void __launch_bounds__(256) ctl_commit_kernel(size_t n, const double* __restrict__ uk, double* __restrict__ u,
                                                          const double* __restrict__ a_new, double* __restrict__ a_prev,
                                                          const double* __restrict__ ctl)
{
    if (__ldcg(ctl + CT_COMMIT) == 0.0) return;
    for (size_t p = (size_t)blockIdx.x * 256 + threadIdx.x; p < n; p += (size_t)gridDim.x * 256) u[p] = uk[p];
    if (__ldcg(ctl + CT_COMMIT_ACC) == 0.0) return;
    for (size_t p = (size_t)blockIdx.x * 256 + threadIdx.x; p < n; p += (size_t)gridDim.x * 256) a_prev[p] = a_new[p];
}

}  // namespace tf
