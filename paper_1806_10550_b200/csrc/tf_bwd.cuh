// tf_bwd.cuh -- back-substitution kernels.
//   ybwd2_* : two-sided y back substitution -> w                                   (S4)
//   xbwd2_* : two-sided x back substitution on the transposed coefficients, then u_{k+1} = u_k + v and
//             res = max|v/u_k|                                                   (S6+S7, (2.21)-(2.22))
//   ybwd_ring_kernel : one-sided back substitution with a cp.async ring (isolated solver of config 4)
// One warp per CTA owns 32 lines; NST stages of line-elements are in flight per warp (TMA boxes + mbarriers,
// or cp.async), so HBM latency is covered by bytes in flight per warp instead of by occupancy.
#pragma once
#include "tf_async.cuh"
#include "tf_tma.cuh"
#include "tf_device.cuh"
#include "tf_partition.cuh"

namespace tf {

template <int NST, int RS, bool VEC>
__global__ void __launch_bounds__(32)
ybwd_ring_kernel(int nx, int ny, const double* __restrict__ al, const double* __restrict__ be,
                 const double* __restrict__ zz, double* __restrict__ w)
{
    extern __shared__ __align__(16) double sm[];           // [NST][3][RS][32]
    const int lane = threadIdx.x;
    const int i0 = blockIdx.x * 32, i = i0 + lane;
    const int cols_ok = min(32, nx - i0);
    const int ntile = (ny + RS - 1) / RS;
    const double* src[3] = {al, be, zz};

    auto issue = [&](int q) {                               // q-th tile from the bottom of the lines
        const int t = ntile - 1 - q;
        if (t >= 0) {
            const int j0 = t * RS, rows_ok = min(RS, ny - j0);
            double* s = sm + (size_t)(q % NST) * 3 * RS * 32;
#pragma unroll
            for (int a = 0; a < 3; ++a)
                warp_copy_block<RS, 32, VEC>(s + a * RS * 32, 32, src[a] + (size_t)j0 * nx + i0, (size_t)nx,
                                             rows_ok, cols_ok, lane);
        }
        cp_async_commit();
    };
#pragma unroll
    for (int q = 0; q < NST - 1; ++q) issue(q);
    double w1 = 0.0, w2 = 0.0;
    for (int q = 0; q < ntile; ++q) {
        cp_async_wait<NST - 2>();
        __syncwarp();
        issue(q + NST - 1);
        const int j0 = (ntile - 1 - q) * RS;
        const double* s = sm + (size_t)(q % NST) * 3 * RS * 32;
#pragma unroll
        for (int r = RS - 1; r >= 0; --r) {
            const int j = j0 + r;
            if (j < ny) {
                const double x = fma(-s[r * 32 + lane], w1, fma(-s[RS * 32 + r * 32 + lane], w2, s[2 * RS * 32 + r * 32 + lane]));
                if (i < nx) w[(size_t)j * nx + i] = x;
                w2 = w1; w1 = x;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Two-sided back substitution (pairs with the two-sided forward kernels of tf_fwd.cuh).
// The forward pass left, for a line x_0 .. x_{N-1} split at mid:
//   k <  mid :  x_k = z_k - al_k x_{k+1} - be_k x_{k+2}        (eliminated from the low end)
//   k >= mid :  x_k = z_k - al_k x_{k-1} - be_k x_{k-2}        (eliminated from the high end)
// The four unknowns around the split, (p,q,r,s) = x_{mid-2}, x_{mid-1}, x_mid, x_{mid+1}, satisfy the rows
// mid-2 .. mid+1 of these relations: a 4x4 system, reduced to 2x2 by substituting p and s.
// ---------------------------------------------------------------------------------------------
struct Join { double p, q, r, s; };

// c[3*k + {0,1,2}] = al, be, z of row mid-2+k
__device__ __forceinline__ Join babe_join(const double* c)
{
    const double a1 = c[0], b1 = c[1], z1 = c[2], a2 = c[3], b2 = c[4], z2 = c[5];
    const double a3 = c[6], b3 = c[7], z3 = c[8], a4 = c[9], b4 = c[10], z4 = c[11];
    const double A11 = fma(-b3, a1, a3), A12 = fma(-b3, b1, 1.0), rA = fma(-b3, z1, z3);
    const double B21 = fma(-b2, b4, 1.0), B22 = fma(-b2, a4, a2), rB = fma(-b2, z4, z2);
    const double det = A11 * B22 - A12 * B21;
    Join J;
    J.q = (rA * B22 - A12 * rB) / det;
    J.r = (A11 * rB - rA * B21) / det;
    J.p = z1 - a1 * J.q - b1 * J.r;
    J.s = z4 - b4 * J.q - a4 * J.r;
    return J;
}

// y direction: coefficient fields [ny][nx], lane <-> column.  grid (ceil(nx/32), 2): blockIdx.y = half.
// CH (partition variant of the isolated solver, tf_partition.cuh step 3): gridDim.z = P chunks, each an independent
// system over rows [lo, hi) split at its own mid; CH = false is the sweep's kernel (lo = 0, hi = ny).
template <int NST, int RS, bool CH = false>
__global__ void __launch_bounds__(32)
ybwd2_tma_kernel(const __grid_constant__ CUtensorMap mA, const __grid_constant__ CUtensorMap mB,
                 const __grid_constant__ CUtensorMap mZ, int nx, int ny, int mid_arg, const double* __restrict__ al,
                 const double* __restrict__ be, const double* __restrict__ zz, double* __restrict__ w, int P = 1,
                 Gate gate = Gate{nullptr, 0.0})
{
    if (gate_closed(gate)) return;
    extern __shared__ unsigned char raw[];
    unsigned char* base = align1024(raw);
    constexpr int BOX = RS * 32;                             // doubles per box
    double* sm = reinterpret_cast<double*>(base);            // [NST][3][RS][32]
    uint64_t* full = reinterpret_cast<uint64_t*>(base + (size_t)NST * 3 * BOX * 8);
    const int lane = threadIdx.x;
    const int i0 = blockIdx.x * 32, i = i0 + lane;
    const int dir = blockIdx.y;
    const bool colok = i < nx;
    const int lo = CH ? chunk_lo(blockIdx.z, P, ny) : 0, hi = CH ? chunk_lo(blockIdx.z + 1, P, ny) : ny;
    const int mid = CH ? chunk_mid(lo, hi) : mid_arg;
    const int nrows = dir ? hi - mid : mid - lo;
    const int ntile = (nrows + RS - 1) / RS;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NST; ++s) mbar_init(full + s, 1);
        mbar_fence_init();
    }
    __syncwarp();
    // first row of the box of the q-th tile in marching order (may be < 0 or reach past ny: TMA zero-fills)
    auto box_row = [&](int q) { return dir ? mid + q * RS : mid - (q + 1) * RS; };
    auto issue = [&](int q) {
        if (q < ntile && lane == 0) {
            const int s = q % NST;
            double* d = sm + (size_t)s * 3 * BOX;
            mbar_expect_tx(full + s, 3 * BOX * 8);
            tma_load_2d(d, &mA, i0, box_row(q), full + s);
            tma_load_2d(d + BOX, &mB, i0, box_row(q), full + s);
            tma_load_2d(d + 2 * BOX, &mZ, i0, box_row(q), full + s);
        }
    };
#pragma unroll
    for (int q = 0; q < NST; ++q) issue(q);
    // interface solve (both halves do it; each keeps the two unknowns on the other side of the split)
    double c12[12];
    {
        const size_t o = (size_t)(mid - 2) * nx + min(i, nx - 1);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            c12[3 * k] = al[o + (size_t)k * nx]; c12[3 * k + 1] = be[o + (size_t)k * nx]; c12[3 * k + 2] = zz[o + (size_t)k * nx];
        }
    }
    const Join J = babe_join(c12);
    double w1 = dir ? J.q : J.r, w2 = dir ? J.p : J.s;
    for (int q = 0; q < ntile; ++q) {
        const int s = q % NST;
        mbar_wait(full + s, (q / NST) & 1);
        const int jb = box_row(q);
        const double* d = sm + (size_t)s * 3 * BOX + lane;
        if (dir == 0) {
            if (jb >= lo) {                                  // full tile: branch-free, one running pointer
                double* wp = w + (size_t)(jb + RS - 1) * nx + i;
#pragma unroll
                for (int r = RS - 1; r >= 0; --r) {
                    const double x = fma(-d[r * 32], w1, fma(-d[BOX + r * 32], w2, d[2 * BOX + r * 32]));
                    st_if(colok, wp, x);
                    wp -= nx;
                    w2 = w1; w1 = x;
                }
            } else {
#pragma unroll
                for (int r = RS - 1; r >= 0; --r) {
                    if (jb + r >= lo) {
                        const double x = fma(-d[r * 32], w1, fma(-d[BOX + r * 32], w2, d[2 * BOX + r * 32]));
                        if (colok) w[(size_t)(jb + r) * nx + i] = x;
                        w2 = w1; w1 = x;
                    }
                }
            }
        } else {
            if (jb + RS <= hi) {
                double* wp = w + (size_t)jb * nx + i;
#pragma unroll
                for (int r = 0; r < RS; ++r) {
                    const double x = fma(-d[r * 32], w1, fma(-d[BOX + r * 32], w2, d[2 * BOX + r * 32]));
                    st_if(colok, wp, x);
                    wp += nx;
                    w2 = w1; w1 = x;
                }
            } else {
#pragma unroll
                for (int r = 0; r < RS; ++r) {
                    if (jb + r < hi) {
                        const double x = fma(-d[r * 32], w1, fma(-d[BOX + r * 32], w2, d[2 * BOX + r * 32]));
                        if (colok) w[(size_t)(jb + r) * nx + i] = x;
                        w2 = w1; w1 = x;
                    }
                }
            }
        }
        __syncwarp();
        issue(q + NST);
    }
}

// Plain fallback of the same two-sided back substitution (any nx, ny; no TMA): lane <-> column, direct loads.
__global__ void __launch_bounds__(32)
ybwd2_plain_kernel(int nx, int ny, int mid, const double* __restrict__ al, const double* __restrict__ be,
                   const double* __restrict__ zz, double* __restrict__ w, Gate gate)
{
    if (gate_closed(gate)) return;
    const int i = blockIdx.x * 32 + threadIdx.x;
    const int dir = blockIdx.y;
    if (i >= nx) return;
    double c12[12];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const size_t o = (size_t)(mid - 2 + k) * nx + i;
        c12[3 * k] = al[o]; c12[3 * k + 1] = be[o]; c12[3 * k + 2] = zz[o];
    }
    const Join J = babe_join(c12);
    double w1 = dir ? J.q : J.r, w2 = dir ? J.p : J.s;
    const int nrows = dir ? ny - mid : mid;
    for (int k = 0; k < nrows; ++k) {
        const size_t o = (size_t)(dir ? mid + k : mid - 1 - k) * nx + i;
        const double x = fma(-al[o], w1, fma(-be[o], w2, zz[o]));
        w[o] = x;
        w2 = w1; w1 = x;
    }
}

// ---------------------------------------------------------------------------------------------
// x direction, two-sided: coefficient fields transposed [nx][ny], lane <-> row j; then S7: u_{k+1} = u_k + v,
// res = max|v/u_k| ((2.21)-(2.22)).  grid (ceil(ny/32), 2): blockIdx.y = half.
// Half 0 marches columns mid-1 .. 0, half 1 columns mid .. nx-1; mid is a multiple of the tile width (16),
// so the u tiles of the two halves (TMA load, in-place update, TMA store) never overlap.
// ---------------------------------------------------------------------------------------------
// UPDATE = true: the sweep's S7 (u tile loaded, updated in place, stored; residual reduced into red).
// UPDATE = false: plain solve, the solution tile is stored through mUout (isolated solver, config 4).
// CH: chunks of columns [lo, hi) as independent systems (see ybwd2_tma_kernel); interior chunk bounds and every mid
// are multiples of the tile width, so tiles of different CTAs stay disjoint.
template <int NST, bool UPDATE, bool CH = false>
__global__ void __launch_bounds__(32)
xbwd2_tma_kernel(const __grid_constant__ CUtensorMap mA, const __grid_constant__ CUtensorMap mB,
                 const __grid_constant__ CUtensorMap mZ, const __grid_constant__ CUtensorMap mUin,
                 const __grid_constant__ CUtensorMap mUout, int nx, int ny, int mid_arg, const double* __restrict__ alT,
                 const double* __restrict__ beT, const double* __restrict__ zzT, double* __restrict__ red, int P = 1,
                 Gate gate = Gate{nullptr, 0.0})
{
    if (gate_closed(gate)) return;
    constexpr int CS = 16;                                   // columns per stage (= one 128-byte swizzled row)
    constexpr int BOX = CS * 32;                             // doubles per coefficient box
    constexpr int STAGE = 4 * BOX * 8;                       // bytes per stage: 3 coefficient boxes + the u tile
    extern __shared__ unsigned char raw[];
    unsigned char* base = align1024(raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(base + (size_t)NST * STAGE);
    const int lane = threadIdx.x;
    const int j0 = blockIdx.x * 32;
    const int dir = blockIdx.y;
    const bool rowok = j0 + lane < ny;
    const int lo = CH ? chunk_lo(blockIdx.z, P, nx) : 0, hi = CH ? chunk_lo(blockIdx.z + 1, P, nx) : nx;
    const int mid = CH ? chunk_mid(lo, hi) : mid_arg;
    const int ncols = dir ? hi - mid : mid - lo;
    const int ntile = (ncols + CS - 1) / CS;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NST; ++s) mbar_init(full + s, 1);
        mbar_fence_init();
    }
    __syncwarp();
    auto tile_col = [&](int q) { return dir ? mid + q * CS : mid - (q + 1) * CS; };
    auto issue = [&](int q) {
        if (q < ntile && lane == 0) {
            const int s = q % NST;
            unsigned char* d = base + (size_t)s * STAGE;
            const int i0 = tile_col(q);
            mbar_expect_tx(full + s, UPDATE ? STAGE : 3 * BOX * 8);
            tma_load_2d(d, &mA, j0, i0, full + s);
            tma_load_2d(d + BOX * 8, &mB, j0, i0, full + s);
            tma_load_2d(d + 2 * BOX * 8, &mZ, j0, i0, full + s);
            if (UPDATE) tma_load_2d(d + 3 * BOX * 8, &mUin, i0, j0, full + s);
        }
    };
#pragma unroll
    for (int q = 0; q < NST - 1; ++q) issue(q);
    double c12[12];
    {
        const size_t o = (size_t)(mid - 2) * ny + min(j0 + lane, ny - 1);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            c12[3 * k] = alT[o + (size_t)k * ny]; c12[3 * k + 1] = beT[o + (size_t)k * ny]; c12[3 * k + 2] = zzT[o + (size_t)k * ny];
        }
    }
    const Join J = babe_join(c12);
    double v1 = dir ? J.q : J.r, v2 = dir ? J.p : J.s;
    double res = 0.0;
    int bad = 0;
    for (int q = 0; q < ntile; ++q) {
        const int s = q % NST;
        mbar_wait(full + s, (q / NST) & 1);
        const int i0 = tile_col(q), cols_ok = min(CS, hi - i0);
        unsigned char* d = base + (size_t)s * STAGE;
        const double* cf = reinterpret_cast<const double*>(d) + lane;
        unsigned char* su = d + 3 * BOX * 8;
        unsigned char* sur = su + lane * 128;                // this lane's swizzled row
        const int sx = (lane & 7) << 4;
        auto pu_of = [&](int c) { return reinterpret_cast<double*>(sur + ((((c >> 1) << 4) ^ sx) + ((c & 1) << 3))); };
        // All shared-memory loads of the tile first, into registers: the in-place update below stores to shared memory,
        // and the compiler must keep every later shared-memory load behind such a store (it cannot prove that the u tile
        // and the coefficient boxes do not alias), which chained load latency + recurrence + store column after column
        // (ncu at 4096^2: 44 % `wait` stalls, 132 cycles per column).
        double A[CS], Bq[CS], Z[CS], U[CS];
#pragma unroll
        for (int c = 0; c < CS; ++c) {
            A[c] = cf[c * 32]; Bq[c] = cf[BOX + c * 32]; Z[c] = cf[2 * BOX + c * 32];
            U[c] = UPDATE ? *pu_of(c) : 0.0;
        }
        auto column = [&](int c) {
            const double v = fma(-A[c], v1, fma(-Bq[c], v2, Z[c]));
            double* pu = pu_of(c);
            if (UPDATE) {
                const double uo = U[c];
                const double un = uo + v;
                const double rr = fabs(v) * rcp(uo);
                res = fmax(res, rowok ? rr : 0.0);           // fmax drops a NaN ratio: bit 1 of `bad` remembers it
                bad |= (rowok && !(un > 0.0 && un <= 1.7976931348623157e308)) ? (un != un ? 3 : 1) : 0;
                *pu = un;
            } else {
                *pu = v;
            }
            v2 = v1; v1 = v;
        };
        if (dir == 0) {                                      // always full tiles (mid is a multiple of CS)
#pragma unroll
            for (int c = CS - 1; c >= 0; --c) column(c);
        } else if (cols_ok == CS) {
#pragma unroll
            for (int c = 0; c < CS; ++c) column(c);
        } else {
#pragma unroll
            for (int c = 0; c < CS; ++c)
                if (c < cols_ok) column(c);
        }
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) {
            tma_store_2d(&mUout, i0, j0, su);
            tma_store_commit();
            tma_store_wait_read<1>();                        // the store of tile q-1 has left shared memory
        }
        __syncwarp();
        issue(q + NST - 1);                                  // refill the stage of tile q-1
    }
    if (lane == 0) tma_store_wait_all<0>();
    if (!UPDATE) return;
    // (2.22) with a NaN winning the max, as in the definition written out: u_k is a finite positive film, so v / u_k is
    // NaN exactly when v is, i.e. exactly when u_k + v is
    if (bad & 2) res = __longlong_as_double(0x7ff8000000000000LL);
    res = warp_max_nonneg(res);
    bad = __any_sync(0xffffffffu, bad);
    if (lane == 0) {
        atomic_max_nonneg(red, res);
        if (bad) atomic_max_nonneg(red + 1, 1.0);
    }
}

// Plain fallback (any nx, ny): thread per row, direct loads (u accesses are strided: correctness path for
// odd or tiny grids, not a fast path).  uk may alias unew.
__global__ void __launch_bounds__(32)
xbwd2_plain_kernel(int nx, int ny, int mid, const double* __restrict__ alT, const double* __restrict__ beT,
                   const double* __restrict__ zzT, const double* uk, double* unew, double* __restrict__ red, Gate gate)
{
    if (gate_closed(gate)) return;
    const int lane = threadIdx.x;
    const int j = blockIdx.x * 32 + lane;
    const int dir = blockIdx.y;
    const bool rowok = j < ny;
    const int jc = min(j, ny - 1);
    double c12[12];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const size_t o = (size_t)(mid - 2 + k) * ny + jc;
        c12[3 * k] = alT[o]; c12[3 * k + 1] = beT[o]; c12[3 * k + 2] = zzT[o];
    }
    const Join J = babe_join(c12);
    double v1 = dir ? J.q : J.r, v2 = dir ? J.p : J.s;
    double res = 0.0;
    int bad = 0;
    const int ncols = dir ? nx - mid : mid;
    for (int k = 0; k < ncols; ++k) {
        const int i = dir ? mid + k : mid - 1 - k;
        const size_t o = (size_t)i * ny + jc;
        const double v = fma(-alT[o], v1, fma(-beT[o], v2, zzT[o]));
        const double uo = uk[(size_t)jc * nx + i];
        const double un = uo + v;
        const double rr = fabs(v) * rcp(uo);
        if (rowok) {
            res = fmax(res, rr);
            bad |= !(un > 0.0 && un <= 1.7976931348623157e308) ? (un != un ? 3 : 1) : 0;
            unew[(size_t)j * nx + i] = un;
        }
        v2 = v1; v1 = v;
    }
    // (2.22) with a NaN winning the max, as in the definition written out: u_k is a finite positive film, so v / u_k is
    // NaN exactly when v is, i.e. exactly when u_k + v is
    if (bad & 2) res = __longlong_as_double(0x7ff8000000000000LL);
    res = warp_max_nonneg(res);
    bad = __any_sync(0xffffffffu, bad);
    if (lane == 0) {
        atomic_max_nonneg(red, res);
        if (bad) atomic_max_nonneg(red + 1, 1.0);
    }
}

}  // namespace tf
