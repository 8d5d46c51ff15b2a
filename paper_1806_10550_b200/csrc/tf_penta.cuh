// tf_penta.cuh -- isolated batched pentadiagonal solve (BASELINE.json config 4).
// Same LU recurrences as the sweeps, with the bands read from memory instead of assembled.
//   dir 1 (systems = columns): lanes along the contiguous index, thread per system, no staging.
//   dir 0 (systems = rows)   : a warp owns 32 rows; 32x32 tiles of the six inputs are loaded coalesced
//                              into padded shared memory and read transposed; the elimination
//                              coefficients are stored transposed, x is written back through a tile.
#pragma once
#include "tf_reduce.cuh"

namespace tf {

// ---- dir 1: forward.  ws = alpha | beta | z, each nrow*ncol, layout [r][c] (as the inputs)
__global__ void __launch_bounds__(32)
penta_col_fwd_kernel(int nrow, int ncol, const double* __restrict__ e, const double* __restrict__ c,
                     const double* __restrict__ d, const double* __restrict__ a, const double* __restrict__ b,
                     const double* __restrict__ y, double* __restrict__ al, double* __restrict__ be,
                     double* __restrict__ zz)
{
    const int s = blockIdx.x * 32 + threadIdx.x;
    if (s >= ncol) return;
    Elim S = {0, 0, 0, 0, 0, 0};
    constexpr int U = 4;
    for (int rb = 0; rb < nrow; rb += U) {
        double E[U], C[U], Dg[U], A[U], B[U], Y[U];
#pragma unroll
        for (int r = 0; r < U; ++r) {
            const size_t o = (size_t)min(rb + r, nrow - 1) * ncol + s;
            E[r] = e[o]; C[r] = c[o]; Dg[r] = d[o]; A[r] = a[o]; B[r] = b[o]; Y[r] = y[o];
        }
#pragma unroll
        for (int r = 0; r < U; ++r) {
            if (rb + r < nrow) {
                double va, vb, vz;
                elim_row(S, E[r], C[r], Dg[r], A[r], B[r], Y[r], va, vb, vz);
                const size_t o = (size_t)(rb + r) * ncol + s;
                al[o] = va; be[o] = vb; zz[o] = vz;
            }
        }
    }
}
// dir 1 backward == ybwd_ring_kernel(nx = ncol, ny = nrow)

// ---- dir 0: forward.  ws arrays are TRANSPOSED: [c][r]
constexpr int PT_ARR = 6;
__global__ void __launch_bounds__(32)
penta_row_fwd_kernel(int nrow, int ncol, const double* __restrict__ e, const double* __restrict__ c,
                     const double* __restrict__ d, const double* __restrict__ a, const double* __restrict__ b,
                     const double* __restrict__ y, double* __restrict__ alT, double* __restrict__ beT,
                     double* __restrict__ zzT)
{
    extern __shared__ double smem[];                       // PT_ARR tiles of XT*XTP
    const double* src[PT_ARR] = {e, c, d, a, b, y};
    const int lane = threadIdx.x;
    const int r0 = blockIdx.x * XT;
    const int row = r0 + lane;
    const bool rowok = row < nrow;
    Elim S = {0, 0, 0, 0, 0, 0};
    const int ntile = (ncol + XT - 1) / XT;
    for (int t = 0; t < ntile; ++t) {
        const int col = t * XT + lane;
        const int cc = col < ncol ? col : ncol - 1;
        __syncwarp();
#pragma unroll
        for (int k = 0; k < PT_ARR; ++k) {
            const double* p = src[k];
            double* sm = smem + k * XT * XTP;
#pragma unroll 8
            for (int rr = 0; rr < XT; ++rr) {
                const int jr = (r0 + rr < nrow) ? r0 + rr : nrow - 1;
                sm[rr * XTP + lane] = p[(size_t)jr * ncol + cc];
            }
        }
        __syncwarp();
        const int nc = min(XT, ncol - t * XT);
        for (int q = 0; q < nc; ++q) {
            const int o = lane * XTP + q;
            double va, vb, vz;
            elim_row(S, smem[o], smem[XT * XTP + o], smem[2 * XT * XTP + o], smem[3 * XT * XTP + o],
                     smem[4 * XT * XTP + o], smem[5 * XT * XTP + o], va, vb, vz);
            if (rowok) {
                const size_t g = (size_t)(t * XT + q) * nrow + row;
                alT[g] = va; beT[g] = vb; zzT[g] = vz;
            }
        }
    }
}

// ---- dir 0: backward; x written through a transposing tile
__global__ void __launch_bounds__(32)
penta_row_bwd_kernel(int nrow, int ncol, const double* __restrict__ alT, const double* __restrict__ beT,
                     const double* __restrict__ zzT, double* __restrict__ x)
{
    __shared__ double sX[XT * XTP];
    const int lane = threadIdx.x;
    const int r0 = blockIdx.x * XT;
    const int row = r0 + lane;
    const int rc = row < nrow ? row : nrow - 1;
    double x1 = 0.0, x2 = 0.0;
    const int ntile = (ncol + XT - 1) / XT;
    for (int t = ntile - 1; t >= 0; --t) {
        const int ihi = min(ncol, (t + 1) * XT) - 1;
        __syncwarp();
        for (int ib = ihi; ib >= t * XT; ib -= PF) {
            double A[PF], B[PF], Z[PF];
#pragma unroll
            for (int r = 0; r < PF; ++r) {
                const size_t o = (size_t)max(ib - r, t * XT) * nrow + rc;
                A[r] = alT[o]; B[r] = beT[o]; Z[r] = zzT[o];
            }
#pragma unroll
            for (int r = 0; r < PF; ++r) {
                const int i = ib - r;
                if (i >= t * XT) {
                    const double v = fma(-A[r], x1, fma(-B[r], x2, Z[r]));
                    sX[lane * XTP + (i - t * XT)] = v;
                    x2 = x1; x1 = v;
                }
            }
        }
        __syncwarp();
        const int col = t * XT + lane;
        if (col < ncol) {
#pragma unroll 8
            for (int rr = 0; rr < XT; ++rr)
                if (r0 + rr < nrow) x[(size_t)(r0 + rr) * ncol + col] = sX[rr * XTP + lane];
        }
    }
}

}  // namespace tf
