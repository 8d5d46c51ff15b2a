// tf_penta.cuh -- isolated batched pentadiagonal solve (BASELINE.json config 4).
// Same LU recurrences as the sweeps, with the bands read from memory instead of assembled.
//   dir 1 (systems = columns): lanes along the contiguous index, thread per system, no staging.
//   dir 0 (systems = rows)   : a warp owns 32 rows; 32x32 tiles of the six inputs are loaded coalesced
//                              into padded shared memory and read transposed; the elimination
//                              coefficients are stored transposed, x is written back through a tile.
#pragma once
#include "tf_reduce.cuh"
#include "tf_tma.cuh"
#include "tf_partition.cuh"

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

// =============================================================================================
// Fast path of the isolated solver (even pitches, lines long enough): the same two-sided elimination and TMA
// rings as the sweeps, with the six band/right-hand-side arrays streamed by TMA instead of assembled.
// Traffic per unknown: 48 B in + 24 B out forward, 24 B in + 8 B out backward = 104 B.
// One warp per CTA; the elimination chain (52 cycles x N/2 rows) is far below the HBM time of these kernels,
// so no producer warps are needed: the marching warp reads its rows straight from the TMA-filled stages.
// =============================================================================================
// ---- systems = columns (lanes along the contiguous index).  grid (ceil(ncol/32), 2), blockIdx.y = half:
// half 0 eliminates rows 0 .. mid-1 downwards, half 1 rows nrow-1 .. mid upwards (reversed system: e<->b, c<->a).
// Coefficients are stored [row][col] like the inputs; ybwd2_tma_kernel / ybwd2_plain_kernel finish the solve.
// Partition variant (tf_partition.cuh step 3): gridDim.z = P chunks, each an independent system over rows [lo, hi)
// whose first two right-hand sides of either march are corrected by the outside unknowns X ([P][4][ncol]).
template <int NST, int RS>
__global__ void __launch_bounds__(32)
penta_col_fwd2_kernel(const __grid_constant__ Maps6 M, int nrow, int ncol, int mid_arg, double* __restrict__ al,
                      double* __restrict__ be, double* __restrict__ zz, int P, const double* __restrict__ X,
                      int Pg = 0, int p_off = 0)
{
    extern __shared__ unsigned char raw[];
    unsigned char* base = align1024(raw);
    constexpr int BOX = RS * 32;                             // doubles per box
    double* sm = reinterpret_cast<double*>(base);            // [NST][6][RS][32]
    uint64_t* full = reinterpret_cast<uint64_t*>(base + (size_t)NST * 6 * BOX * 8);
    const int lane = threadIdx.x;
    const int i0 = blockIdx.x * 32, i = i0 + lane;
    const int dir = blockIdx.y, p = blockIdx.z;
    const int colok = i < ncol ? 1 : 0;
    const int lo = chunk_lo(p, P, nrow), hi = chunk_lo(p + 1, P, nrow);
    const int mid = P > 1 ? chunk_mid(lo, hi) : mid_arg;
    const int jmin = dir ? mid : lo, jmax = dir ? hi : mid;
    const int nrows = jmax - jmin;
    double xfar = 0.0, xnear = 0.0;                          // known unknowns just outside this march's first row
    if (Pg == 0) Pg = P;                                     // single device; else local chunk p is chunk p_off + p of Pg
    const int pg = p_off + p;
    if (Pg > 1 && (dir ? pg < Pg - 1 : pg > 0)) {
        const double* xo = X + (size_t)(dir ? (pg + 1) * 4 : (pg - 1) * 4 + 2) * ncol + min(i, ncol - 1);
        xfar = dir ? xo[ncol] : xo[0];
        xnear = dir ? xo[0] : xo[ncol];
    }
    const int ntile = (nrows + RS - 1) / RS;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NST; ++s) mbar_init(full + s, 1);
        mbar_fence_init();
    }
    __syncwarp();
    auto box_row = [&](int q) { return dir ? hi - (q + 1) * RS : lo + q * RS; };
    auto issue = [&](int q) {
        if (q < ntile && lane == 0) {
            const int s = q % NST;
            double* d = sm + (size_t)s * 6 * BOX;
            mbar_expect_tx(full + s, 6 * BOX * 8);
#pragma unroll
            for (int k = 0; k < 6; ++k) tma_load_2d(d + k * BOX, &M.m[k], i0, box_row(q), full + s);
        }
    };
#pragma unroll
    for (int q = 0; q < NST; ++q) issue(q);
    Elim2 S = elim2_init();
    const ptrdiff_t step = dir ? -(ptrdiff_t)ncol : (ptrdiff_t)ncol;
    ptrdiff_t o = (ptrdiff_t)(dir ? hi : lo - 1) * ncol + i;   // the row before the first one
    const int oe = dir ? 4 * BOX : 0, oc = dir ? 3 * BOX : BOX, oa = dir ? BOX : 3 * BOX, ob = dir ? 0 : 4 * BOX;
    int k = 0;                                               // rows eliminated so far
    for (int q = 0; q < ntile; ++q) {
        const int s = q % NST;
        mbar_wait(full + s, (q / NST) & 1);
        const int jb = box_row(q);
        const double* d = sm + (size_t)s * 6 * BOX + lane;
        if (jb >= jmin && jb + RS <= jmax && q > 0) {
#pragma unroll
            for (int rr = 0; rr < RS; ++rr) {
                const int r = dir ? RS - 1 - rr : rr;
                double va, vb, vz;
                elim2_row(S, d[oe + r * 32], d[oc + r * 32], d[2 * BOX + r * 32], d[oa + r * 32], d[ob + r * 32],
                          d[5 * BOX + r * 32], va, vb, vz);
                st3_if(colok, al + o, va, be + o, vb, zz + o, vz);
                o += step;
            }
            k += RS;
        } else {
            for (int rr = 0; rr < RS; ++rr) {
                const int r = dir ? RS - 1 - rr : rr;
                const int j = jb + r;
                if (j >= jmin && j < jmax) {
                    double va, vb, vz;
                    const double ve = d[oe + r * 32], vc = d[oc + r * 32];
                    double vy = d[5 * BOX + r * 32];
                    if (k == 0) vy -= ve * xfar + vc * xnear;
                    if (k == 1) vy -= ve * xnear;
                    elim2_row(S, ve, vc, d[2 * BOX + r * 32], d[oa + r * 32], d[ob + r * 32], vy, va, vb, vz);
                    st3_if(colok && k > 0, al + o, va, be + o, vb, zz + o, vz);
                    o += step;
                    ++k;
                }
            }
        }
        __syncwarp();
        issue(q + NST);
    }
    double va, vb, vz;
    elim2_flush(S, va, vb, vz);
    st3_if(colok, al + o, va, be + o, vb, zz + o, vz);
}

// ---- systems = rows (contiguous).  lane <-> row of a block of 32 rows, marching along the columns through
// [32 rows x 16 cols] TMA boxes with the 128-byte swizzle (conflict-free column reads); coefficients are stored
// TRANSPOSED [col][row] (coalesced).  grid (ceil(nrow/32), 2): half 0 columns 0 .. mid-1 ascending, half 1
// columns ncol-1 .. mid descending.  xbwd2_tma_kernel<.., false> / penta_row_bwd2_plain_kernel finish the solve.
// Partition variant: gridDim.z = P chunks of columns [lo, hi), X = [P][4][nrow] (see penta_col_fwd2_kernel).
template <int NST>
__global__ void __launch_bounds__(32)
penta_row_fwd2_kernel(const __grid_constant__ Maps6 M, int nrow, int ncol, int mid_arg, double* __restrict__ alT,
                      double* __restrict__ beT, double* __restrict__ zzT, int P, const double* __restrict__ X,
                      int Pg = 0, int p_off = 0)
{
    constexpr int CS = 16;
    constexpr int TILE = 32 * CS * 8;                        // bytes per array tile (4 KiB, 1024-aligned)
    extern __shared__ unsigned char raw[];
    unsigned char* base = align1024(raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(base + (size_t)NST * 6 * TILE);
    const int lane = threadIdx.x;
    const int r0 = blockIdx.x * 32;
    const int dir = blockIdx.y, p = blockIdx.z;
    const int rowok = r0 + lane < nrow ? 1 : 0;
    const int lo = chunk_lo(p, P, ncol), hi = chunk_lo(p + 1, P, ncol);
    const int mid = P > 1 ? chunk_mid(lo, hi) : mid_arg;
    const int imin = dir ? mid : lo, imax = dir ? hi : mid;
    double xfar = 0.0, xnear = 0.0;
    if (Pg == 0) Pg = P;
    const int pg = p_off + p;
    if (Pg > 1 && (dir ? pg < Pg - 1 : pg > 0)) {
        const double* xo = X + (size_t)(dir ? (pg + 1) * 4 : (pg - 1) * 4 + 2) * nrow + min(r0 + lane, nrow - 1);
        xfar = dir ? xo[nrow] : xo[0];
        xnear = dir ? xo[0] : xo[nrow];
    }
    const int ncols = imax - imin;
    const int ntile = (ncols + CS - 1) / CS;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NST; ++s) mbar_init(full + s, 1);
        mbar_fence_init();
    }
    __syncwarp();
    auto tile_col = [&](int q) { return dir ? hi - (q + 1) * CS : lo + q * CS; };
    auto issue = [&](int q) {
        if (q < ntile && lane == 0) {
            const int s = q % NST;
            unsigned char* d = base + (size_t)s * 6 * TILE;
            mbar_expect_tx(full + s, 6 * TILE);
#pragma unroll
            for (int k = 0; k < 6; ++k) tma_load_2d(d + k * TILE, &M.m[k], tile_col(q), r0, full + s);
        }
    };
#pragma unroll
    for (int q = 0; q < NST; ++q) issue(q);
    Elim2 S = elim2_init();
    const ptrdiff_t step = dir ? -(ptrdiff_t)nrow : (ptrdiff_t)nrow;
    ptrdiff_t o = (ptrdiff_t)(dir ? hi : lo - 1) * nrow + r0 + lane;
    const int oe = dir ? 4 * TILE : 0, oc = dir ? 3 * TILE : TILE, oa = dir ? TILE : 3 * TILE, ob = dir ? 0 : 4 * TILE;
    const int sx = (lane & 7) << 4;
    int k = 0;
    for (int q = 0; q < ntile; ++q) {
        const int s = q % NST;
        mbar_wait(full + s, (q / NST) & 1);
        const int ib = tile_col(q);
        const unsigned char* d = base + (size_t)s * 6 * TILE + lane * 128;     // this lane's swizzled row
        auto at = [&](int off, int c) {
            return *reinterpret_cast<const double*>(d + off + ((((c >> 1) << 4) ^ sx) + ((c & 1) << 3)));
        };
        if (ib >= imin && ib + CS <= imax && q > 0) {
#pragma unroll
            for (int cc = 0; cc < CS; ++cc) {
                const int c = dir ? CS - 1 - cc : cc;
                double va, vb, vz;
                elim2_row(S, at(oe, c), at(oc, c), at(2 * TILE, c), at(oa, c), at(ob, c), at(5 * TILE, c), va, vb, vz);
                st3_if(rowok, alT + o, va, beT + o, vb, zzT + o, vz);
                o += step;
            }
            k += CS;
        } else {
            for (int cc = 0; cc < CS; ++cc) {
                const int c = dir ? CS - 1 - cc : cc;
                const int i = ib + c;
                if (i >= imin && i < imax) {
                    double va, vb, vz;
                    const double ve = at(oe, c), vc = at(oc, c);
                    double vy = at(5 * TILE, c);
                    if (k == 0) vy -= ve * xfar + vc * xnear;
                    if (k == 1) vy -= ve * xnear;
                    elim2_row(S, ve, vc, at(2 * TILE, c), at(oa, c), at(ob, c), vy, va, vb, vz);
                    st3_if(rowok && k > 0, alT + o, va, beT + o, vb, zzT + o, vz);
                    o += step;
                    ++k;
                }
            }
        }
        __syncwarp();
        issue(q + NST);
    }
    double va, vb, vz;
    elim2_flush(S, va, vb, vz);
    st3_if(rowok, alT + o, va, beT + o, vb, zzT + o, vz);
}

}  // namespace tf
