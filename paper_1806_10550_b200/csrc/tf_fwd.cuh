// tf_fwd.cuh -- warp-specialised forward kernels (assembly + LU forward elimination), S1-S6 forward halves.
//
// Why: a sweep has only nx (ny) independent lines = 256 warps at 8192^2 for 592 SM sub-partitions, and the
// assembly of one matrix row costs ~100 fp64 instructions against ~20 for the elimination recurrence.  If
// the thread that carries the recurrence also assembles, under half of the fp64 pipes are ever busy and
// the serial chain is 5x longer than it must be.  So a CTA owns one strip of lines and splits the work:
//   * NP producer warps assemble rows (bands A,c,q,a and right-hand side R) for disjoint row chunks of a
//     tile -- embarrassingly parallel -- and hand them over through a shared-memory ring;
//   * 1 consumer warp runs the pentadiagonal recurrence and streams alpha,beta,z out.
// Hand-over is by mbarriers (full/empty per stage), no __syncthreads in the steady state.
#pragma once
#include "tf_device.cuh"
#include "tf_tma.cuh"

namespace tf {

constexpr int YW_VALID = 28;     // columns per strip (lanes 2..29; lanes 0,1,30,31 are x-halo)

// rolling state of a thread marching down a column (see yfwd_kernel in tf_sweeps.cuh for the same scheme)
struct YState {
    double hm1, h0, hp1;         // h(j-1), h(j), h(j+1)
    double hR0;                  // h(j)[i+1]
    Cell c0;                     // cell (j)
    double L0;                   // lap h (j)
    Face fm;                     // face j-1/2 (folded / zeroed)
    double phim;                 // s*Fy(j-1/2)/dy
};

// MODE 0: bring in cell (j+1) only;  1: also face j+1/2;  2: also produce row j (bands + R).
// out5 = {A_{j+1/2}, c, q, a, R}
// INTERIOR: all faces touched are interior and unfolded (1 <= j <= ny-3): no boundary logic at all.
template <int N, int M, int MODE, bool INTERIOR>
__device__ __forceinline__ void y_advance(YState& S, int j, double hp2, const Params& P, const Dir& DX, const Dir& DY,
                                          bool xface, double rhs_in, double* out5, double& sD_out)
{
    const unsigned FULL = 0xffffffffu;
    const int ny = P.ny;
    const double hL = __shfl_up_sync(FULL, S.hp1, 1), hR = __shfl_down_sync(FULL, S.hp1, 1);
    const double Lp = fma((hL + hR) - 2.0 * S.hp1, P.rdx2, ((hp2 + S.h0) - 2.0 * S.hp1) * P.rdy2);
    const Cell cp = cell_functions<N, M>(S.hp1, P);
    Face fp = {0.0, 0.0, 0.0};
    double phip = 0.0;
    if (MODE >= 1) {
        const bool yface = (j >= 0) && (j <= ny - 2);
        const double dh = S.hp1 - S.h0;
        const double sf0 = S.c0.f0 + cp.f0, sf1 = S.c0.f1 + cp.f1;
        fp = face_partials(S.hm1, hp2, dh, sf0, sf1, S.c0, cp, DY);
        phip = DY.cb * fma(sf0, Lp - S.L0, sf1 * dh);
        if (!INTERIOR) {
            if (j == 0) fp.p1 -= fp.A;
            if (j == ny - 2) fp.p2 += fp.A;
            if (!yface) { fp.A = 0.0; fp.p1 = 0.0; fp.p2 = 0.0; phip = 0.0; }
        }
    }
    if (MODE == 2) {
        const double f0R = __shfl_down_sync(FULL, S.c0.f0, 1), f1R = __shfl_down_sync(FULL, S.c0.f1, 1);
        const double LR = __shfl_down_sync(FULL, S.L0, 1);
        double phixp = DX.cb * fma(S.c0.f0 + f0R, LR - S.L0, (S.c0.f1 + f1R) * (S.hR0 - S.h0));
        if (!xface) phixp = 0.0;
        const double phixm = __shfl_up_sync(FULL, phixp, 1);
        const double sD = (phixp - phixm) + (phip - S.phim);
        sD_out = sD;
        out5[0] = fp.A;
        out5[1] = -fp.A - S.fm.p1;
        out5[2] = 1.0 + fp.p1 - S.fm.p2;
        out5[3] = fp.p2 - S.fm.A;
        out5[4] = (rhs_in - S.h0) - sD;            // FIRST: caller passes rhs_in = b, fixed up below
    }
    S.hm1 = S.h0; S.h0 = S.hp1; S.hp1 = hp2; S.hR0 = hR;
    S.c0 = cp; S.L0 = Lp;
    if (MODE >= 1) { S.fm = fp; S.phim = phip; }
}

template <int N, int M, bool FIRST, int NP, int RP, int NSTG>
__global__ void __launch_bounds__(32 * (NP + 1))
yfwd_ws_kernel(Params P, Dir DX, Dir DY, const double* __restrict__ u, double* __restrict__ bn,
               double* __restrict__ al, double* __restrict__ be, double* __restrict__ zz)
{
    constexpr int RT = NP * RP;                       // rows per tile / stage
    constexpr int SV = RT * 32;                       // doubles per value plane of a stage
    extern __shared__ __align__(16) unsigned char raw[];
    double* sm = reinterpret_cast<double*>(raw);      // [NSTG][5][RT][32]
    uint64_t* full = reinterpret_cast<uint64_t*>(raw + (size_t)NSTG * 5 * SV * 8);
    uint64_t* empty = full + NSTG;
    const int nx = P.nx, ny = P.ny;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NSTG; ++s) { mbar_init(full + s, NP); mbar_init(empty + s, 1); }
        mbar_fence_init();
    }
    __syncthreads();
    const int i = blockIdx.x * YW_VALID - 2 + lane;
    const int ntile = (ny + RT - 1) / RT;

    if (warp < NP) {
        // ------------------------------------------------------------------ producer: rows [j0, j0+RP) of each tile
        const int ic = ghost(i, nx);
        const bool xface = (i >= 0) && (i <= nx - 2);
        const bool outl = (lane >= 2) && (lane < 2 + YW_VALID) && (i < nx);
        const double* up = u + ic;
        const double* bp = bn + ic;
        for (int t = 0; t < ntile; ++t) {
            const int s = t % NSTG;
            const int j0 = t * RT + warp * RP;
            const bool interior = (j0 >= 2) && (j0 + RP + 1 <= ny - 2);
            double hq[RP + 4], bq[RP];
            if (interior) {
                const double* hp = up + (size_t)(j0 - 2) * nx;
#pragma unroll
                for (int k = 0; k < RP + 4; ++k) hq[k] = hp[(size_t)k * nx];
                const double* bq0 = bp + (size_t)j0 * nx;
#pragma unroll
                for (int k = 0; k < RP; ++k) bq[k] = FIRST ? 0.0 : bq0[(size_t)k * nx];
            } else if (j0 < ny) {
#pragma unroll
                for (int k = 0; k < RP + 4; ++k) hq[k] = up[(size_t)ghost(j0 - 2 + k, ny) * nx];
#pragma unroll
                for (int k = 0; k < RP; ++k) bq[k] = FIRST ? 0.0 : bp[(size_t)clampi(j0 + k, 0, ny - 1) * nx];
            }
            mbar_wait(empty + s, ((t / NSTG) & 1) ^ 1);
            double* st = sm + (size_t)s * 5 * SV + (warp * RP) * 32 + lane;
            YState S;
            S.hm1 = 0.0; S.h0 = hq[0]; S.hp1 = hq[1]; S.hR0 = 0.0;
            S.c0 = {0, 0, 0, 0}; S.L0 = 0.0; S.fm = {0, 0, 0}; S.phim = 0.0;
            double o5[5], sD;
            if (interior) {
                y_advance<N, M, 0, true>(S, j0 - 2, hq[2], P, DX, DY, xface, 0.0, o5, sD);
                y_advance<N, M, 1, true>(S, j0 - 1, hq[3], P, DX, DY, xface, 0.0, o5, sD);
                double* bo = bn + (size_t)j0 * nx + i;
#pragma unroll
                for (int r = 0; r < RP; ++r) {
                    const double hcur = S.h0;
                    y_advance<N, M, 2, true>(S, j0 + r, hq[r + 4], P, DX, DY, xface, FIRST ? hcur : bq[r], o5, sD);
                    if (FIRST) {
                        const double b = hcur - sD;
                        if (outl) bo[(size_t)r * nx] = b;
                        o5[4] = (b - hcur) - sD;
                    }
#pragma unroll
                    for (int v = 0; v < 5; ++v) st[v * SV + r * 32] = o5[v];
                }
            } else if (j0 < ny) {
                y_advance<N, M, 0, false>(S, j0 - 2, hq[2], P, DX, DY, xface, 0.0, o5, sD);
                y_advance<N, M, 1, false>(S, j0 - 1, hq[3], P, DX, DY, xface, 0.0, o5, sD);
#pragma unroll
                for (int r = 0; r < RP; ++r) {
                    const int j = j0 + r;
                    if (j < ny) {
                        const double hcur = S.h0;
                        y_advance<N, M, 2, false>(S, j, hq[r + 4], P, DX, DY, xface, FIRST ? hcur : bq[r], o5, sD);
                        if (FIRST) {
                            const double b = hcur - sD;
                            if (outl) bn[(size_t)j * nx + i] = b;
                            o5[4] = (b - hcur) - sD;
                        }
#pragma unroll
                        for (int v = 0; v < 5; ++v) st[v * SV + r * 32] = o5[v];
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(full + s);
        }
    } else {
        // ------------------------------------------------------------------ consumer: the recurrence
        const bool outl = (lane >= 2) && (lane < 2 + YW_VALID) && (i < nx);
        Elim S = {0, 0, 0, 0, 0, 0};
        double e = 0.0;
        for (int t = 0; t < ntile; ++t) {
            const int s = t % NSTG;
            mbar_wait(full + s, (t / NSTG) & 1);
            const double* st = sm + (size_t)s * 5 * SV + lane;
            const int jt = t * RT;
            const int nrow = min(RT, ny - jt);
            size_t o = (size_t)jt * nx + i;
            if (nrow == RT) {
#pragma unroll 8
                for (int r = 0; r < RT; ++r) {
                    const double A = st[r * 32], c = st[SV + r * 32], q = st[2 * SV + r * 32], a = st[3 * SV + r * 32];
                    const double R = st[4 * SV + r * 32];
                    double va, vb, vz;
                    elim_row(S, e, c, q, a, A, R, va, vb, vz);
                    e = A;
                    if (outl) { al[o] = va; be[o] = vb; zz[o] = vz; }
                    o += nx;
                }
            } else {
                for (int r = 0; r < nrow; ++r) {
                    const double A = st[r * 32], c = st[SV + r * 32], q = st[2 * SV + r * 32], a = st[3 * SV + r * 32];
                    const double R = st[4 * SV + r * 32];
                    double va, vb, vz;
                    elim_row(S, e, c, q, a, A, R, va, vb, vz);
                    e = A;
                    if (outl) { al[o] = va; be[o] = vb; zz[o] = vz; }
                    o += nx;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + s);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// x forward, warp-specialised.  A CTA owns 32 rows.  Producers work with lanes ALONG the lines (lane <->
// column i, coalesced loads, neighbours by shuffle; only x-neighbours are needed) and write
// the bands transposed into the stage ([column][33]: conflict-free both ways); the consumer has
// lane <-> row and marches i = 0..nx-1.  Coefficients go out transposed ([i][j]) so the stores are
// coalesced too.  Tile = 28 columns (32 lanes minus 2 halo lanes each side).
// ---------------------------------------------------------------------------------------------
constexpr int XW_CT = 28;
constexpr int XW_LD = 33;

template <int N, int M, int NP, int NSTG>
__global__ void __launch_bounds__(32 * (NP + 1))
xfwd_ws_kernel(Params P, Dir DX, const double* __restrict__ u, const double* __restrict__ w,
               double* __restrict__ alT, double* __restrict__ beT, double* __restrict__ zzT)
{
    constexpr int SV = XW_CT * XW_LD;                 // doubles per value plane of a stage
    extern __shared__ __align__(16) unsigned char raw[];
    double* sm = reinterpret_cast<double*>(raw);      // [NSTG][5][CT][33]
    uint64_t* full = reinterpret_cast<uint64_t*>(raw + (size_t)NSTG * 5 * SV * 8);
    uint64_t* empty = full + NSTG;
    const unsigned FULL = 0xffffffffu;
    const int nx = P.nx, ny = P.ny;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NSTG; ++s) { mbar_init(full + s, NP); mbar_init(empty + s, 1); }
        mbar_fence_init();
    }
    __syncthreads();
    const int j0 = blockIdx.x * 32;
    const int ntile = (nx + XW_CT - 1) / XW_CT;

    if (warp < NP) {
        // ------------------------------------------------------------------ producer: rows warp, warp+NP, ...
        for (int t = 0; t < ntile; ++t) {
            const int s = t % NSTG;
            const int i = t * XW_CT - 2 + lane;
            const int ic = ghost(i, nx);
            const bool face_ok = (i >= 0) && (i <= nx - 2);
            const bool col_ok = (lane >= 2) && (lane < 2 + XW_CT) && (i < nx);
            constexpr int NR = 32 / NP;
            double hq[NR], wq[NR];
#pragma unroll
            for (int k = 0; k < NR; ++k) {
                const int jr = min(j0 + warp + k * NP, ny - 1);
                hq[k] = u[(size_t)jr * nx + ic];
                wq[k] = col_ok ? w[(size_t)jr * nx + i] : 0.0;
            }
            mbar_wait(empty + s, ((t / NSTG) & 1) ^ 1);
            double* st = sm + (size_t)s * 5 * SV + (lane - 2) * XW_LD;
#pragma unroll
            for (int k = 0; k < NR; ++k) {
                const int r = warp + k * NP;
                const double h0 = hq[k];
                const double hm1 = __shfl_up_sync(FULL, h0, 1);
                const double hp1 = __shfl_down_sync(FULL, h0, 1), hp2 = __shfl_down_sync(FULL, h0, 2);
                const Cell c0 = cell_functions<N, M>(h0, P);
                Cell c1;
                c1.f0 = __shfl_down_sync(FULL, c0.f0, 1); c1.f1 = __shfl_down_sync(FULL, c0.f1, 1);
                c1.g0 = __shfl_down_sync(FULL, c0.g0, 1); c1.g1 = __shfl_down_sync(FULL, c0.g1, 1);
                Face fp = face_partials(hm1, hp2, hp1 - h0, c0.f0 + c1.f0, c0.f1 + c1.f1, c0, c1, DX);
                if (i == 0) fp.p1 -= fp.A;
                if (i == nx - 2) fp.p2 += fp.A;
                if (!face_ok) { fp.A = 0.0; fp.p1 = 0.0; fp.p2 = 0.0; }
                Face fm;
                fm.A = __shfl_up_sync(FULL, fp.A, 1); fm.p1 = __shfl_up_sync(FULL, fp.p1, 1);
                fm.p2 = __shfl_up_sync(FULL, fp.p2, 1);
                if (col_ok) {
                    st[r] = fp.A;
                    st[SV + r] = -fp.A - fm.p1;
                    st[2 * SV + r] = 1.0 + fp.p1 - fm.p2;
                    st[3 * SV + r] = fp.p2 - fm.A;
                    st[4 * SV + r] = wq[k];
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(full + s);
        }
    } else {
        // ------------------------------------------------------------------ consumer: lane <-> row j0 + lane
        const int j = j0 + lane;
        const bool rowok = j < ny;
        Elim S = {0, 0, 0, 0, 0, 0};
        double e = 0.0;
        for (int t = 0; t < ntile; ++t) {
            const int s = t % NSTG;
            mbar_wait(full + s, (t / NSTG) & 1);
            const double* st = sm + (size_t)s * 5 * SV + lane;
            const int i0 = t * XW_CT;
            const int ncol = min(XW_CT, nx - i0);
            size_t o = (size_t)i0 * ny + j;
            for (int c = 0; c < ncol; ++c) {
                const double A = st[c * XW_LD], cc = st[SV + c * XW_LD], q = st[2 * SV + c * XW_LD];
                const double a = st[3 * SV + c * XW_LD], R = st[4 * SV + c * XW_LD];
                double va, vb, vz;
                elim_row(S, e, cc, q, a, A, R, va, vb, vz);
                e = A;
                if (rowok) { alT[o] = va; beT[o] = vb; zzT[o] = vz; }
                o += ny;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + s);
        }
    }
}

}  // namespace tf
