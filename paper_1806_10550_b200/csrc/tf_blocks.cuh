// tf_blocks.cuh -- pack / unpack of rectangular blocks of a field for the exchange steps of the distributed time step
// (SURVEY.md 8(e)): one kernel gathers every block a rank sends into the contiguous all-to-all
// buffer, one kernel scatters what it received into the destination field and, in the same pass, fills the ghost
// columns of a halo'd column block that lies at a domain edge by the reflection of (2.28)
// (h_{-1} = h_0, h_{-2} = h_1, h_{nx} = h_{nx-1}, h_{nx+1} = h_{nx-2}).  Memory movement only, 16 B/pt per direction.
#pragma once
#include <cuda_runtime.h>

namespace tf {

constexpr int BLK_MAX = 64;          // blocks per call (= ranks of the group)
constexpr int BLK_THREADS = 256;
constexpr int BLK_ROWS = 8;          // rows per CTA

struct Rect { int row0, nrows, col0, ncols; long long off; };
struct Rects { Rect r[BLK_MAX]; int n; };

// buf[off + row * ncols + col] = field[(row0 + row) * ld + col0 + col]
__global__ void __launch_bounds__(BLK_THREADS)
blocks_gather_kernel(const double* __restrict__ field, int ld, const __grid_constant__ Rects R, double* __restrict__ buf)
{
    const Rect q = R.r[blockIdx.z];
    const int rlo = blockIdx.y * BLK_ROWS;
    if (rlo >= q.nrows) return;
    const int rhi = min(rlo + BLK_ROWS, q.nrows);
    for (int c = blockIdx.x * BLK_THREADS + threadIdx.x; c < q.ncols; c += gridDim.x * BLK_THREADS)
        for (int r = rlo; r < rhi; ++r)
            buf[q.off + (long long)r * q.ncols + c] = field[(size_t)(q.row0 + r) * ld + q.col0 + c];
}

// the reverse; lrefl: columns 1, 0 of the field are the ghosts of columns 2, 3; rrefl >= 0: columns rrefl, rrefl + 1
// are the ghosts of columns rrefl - 1, rrefl - 2
__global__ void __launch_bounds__(BLK_THREADS)
blocks_scatter_kernel(const double* __restrict__ buf, const __grid_constant__ Rects R, double* __restrict__ field, int ld,
                      int lrefl, int rrefl)
{
    const Rect q = R.r[blockIdx.z];
    const int rlo = blockIdx.y * BLK_ROWS;
    if (rlo >= q.nrows) return;
    const int rhi = min(rlo + BLK_ROWS, q.nrows);
    for (int c = blockIdx.x * BLK_THREADS + threadIdx.x; c < q.ncols; c += gridDim.x * BLK_THREADS) {
        const int col = q.col0 + c;
        // ghost columns that mirror this one, if any (a block of one or two own columns feeds both sides)
        const int gl = (lrefl && (col == 2 || col == 3)) ? 3 - col : -1;
        const int gr = (rrefl >= 0 && (col == rrefl - 1 || col == rrefl - 2)) ? 2 * rrefl - 1 - col : -1;
        for (int r = rlo; r < rhi; ++r) {
            const double v = buf[q.off + (long long)r * q.ncols + c];
            double* row = field + (size_t)(q.row0 + r) * ld;
            row[col] = v;
            if (gl >= 0) row[gl] = v;
            if (gr >= 0) row[gr] = v;
        }
    }
}

// One block straight from field to field (the part of an exchange a rank keeps for itself never enters the
// all-to-all buffers): dst[(drow0 + r) * dld + dcol0 + c] = src[(srow0 + r) * sld + scol0 + c], ghosts as above.
__global__ void __launch_bounds__(BLK_THREADS)
block_copy_kernel(const double* __restrict__ src, int sld, int srow0, int scol0, double* __restrict__ dst, int dld,
                  int drow0, int dcol0, int nrows, int ncols, int lrefl, int rrefl)
{
    const int rlo = blockIdx.y * BLK_ROWS;
    const int rhi = min(rlo + BLK_ROWS, nrows);
    for (int c = blockIdx.x * BLK_THREADS + threadIdx.x; c < ncols; c += gridDim.x * BLK_THREADS) {
        const int col = dcol0 + c;
        const int gl = (lrefl && (col == 2 || col == 3)) ? 3 - col : -1;
        const int gr = (rrefl >= 0 && (col == rrefl - 1 || col == rrefl - 2)) ? 2 * rrefl - 1 - col : -1;
        for (int r = rlo; r < rhi; ++r) {
            const double v = src[(size_t)(srow0 + r) * sld + scol0 + c];
            double* row = dst + (size_t)(drow0 + r) * dld;
            row[col] = v;
            if (gl >= 0) row[gl] = v;
            if (gr >= 0) row[gr] = v;
        }
    }
}

// Residual record {res, bad} of one iteration before it is max-reduced over the ranks: a NaN must win the max (it
// would be dropped by it) and must close the gates of the iterations launched ahead, so it becomes +inf with bad = 1.
__global__ void record_sanitize_kernel(double* rec)
{
    const double r = rec[0];
    if (r != r || r == __longlong_as_double(0x7ff0000000000000LL)) {
        rec[0] = __longlong_as_double(0x7ff0000000000000LL);
        rec[1] = 1.0;
    }
}

}  // namespace tf
