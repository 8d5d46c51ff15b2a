// tf_sweeps.cuh -- the four kernels of one pseudo-Newton iteration ((2.19)-(2.21)):
//   yfwd : S1+S2+S3 + forward half of S4   (assemble R and I+sJ_y on the fly, eliminate)   thread per column
//   ybwd : back substitution of S4 -> w                                                     thread per column
//   xfwd : S1+S5 + forward half of S6      (assemble I+sJ_x, eliminate)                     thread per row, smem-transposed tiles
//   xbwd : back substitution of S6 + S7    (u_{k+1} = u_k + v, res = max|v/u_k|)            thread per row
// Fields are row-major [j][i].  The elimination coefficients (alpha, beta, z) of the y-sweep are
// stored [j][i]; those of the x-sweep are stored TRANSPOSED [i][j], so both are written and
// read with lanes along the contiguous index (coalesced) without staging.
#pragma once
#include "tf_device.cuh"

namespace tf {

constexpr int YF_VALID = 28;   // columns a 32-lane warp produces in yfwd (2 halo lanes each side)
constexpr int PF = 8;          // rows of register prefetch in the marching kernels

// ---------------------------------------------------------------------------------------------
// y forward.  Lane l of block b owns column i = 28 b - 2 + l and marches j = 0..ny-1 with a rolling
// register window: h(j-1..j+2), cells (f0,f1,f0',f1',lap) of rows j, j+1, the face j-1/2.
// x-neighbours come from the adjacent lanes by shuffle; lanes 0,1,30,31 are halo (results unused).
// FIRST = first Newton iteration of a time step: u_k = u^n, so b^n = u - sD(u) is produced here
// (b^n "only computed at the initial iteration step") and R = (b^n - u) - sD(u).
// ---------------------------------------------------------------------------------------------
template <int N, int M, bool FIRST>
__global__ void __launch_bounds__(32)
yfwd_kernel(Params P, Dir DX, Dir DY, const double* __restrict__ u, double* __restrict__ bn,
            double* __restrict__ al, double* __restrict__ be, double* __restrict__ zz)
{
    const unsigned FULL = 0xffffffffu;
    const int nx = P.nx, ny = P.ny;
    const int lane = threadIdx.x;
    const int i = blockIdx.x * YF_VALID - 2 + lane;
    const int ic = ghost(i, nx);
    const bool xface = (i >= 0) && (i <= nx - 2);            // face i+1/2 is interior
    const bool outl = (lane >= 2) && (lane < 2 + YF_VALID) && (i < nx);
    const double* up = u + ic;
    const double* bp = bn + ic;

    // window before step j = -1:  h(-2) = h[1], h(-1) = h[0], h(0) = h[0]
    double hm1 = up[(size_t)1 * nx], h0 = up[0], hp1 = h0;
    double hR0 = 0.0;                                      // h(j)[i+1]
    Cell c0 = {0, 0, 0, 0}, cp;                            // cells of rows j, j+1
    double L0 = 0.0, Lp;
    Face fm = {0, 0, 0};                                   // face j-1/2 (folded)
    double phim = 0.0;                                     // s*Fy(j-1/2)/dy
    Elim S = {0, 0, 0, 0, 0, 0};

    double hq[PF], bq[PF];
#pragma unroll
    for (int r = 0; r < PF; ++r) {
        hq[r] = up[(size_t)ghost(-1 + r + 2, ny) * nx];
        bq[r] = FIRST ? 0.0 : bp[(size_t)clampi(-1 + r, 0, ny - 1) * nx];
    }
    for (int jb = -1; jb < ny; jb += PF) {
        double hn[PF], bnn[PF];
#pragma unroll
        for (int r = 0; r < PF; ++r) {
            hn[r] = up[(size_t)ghost(jb + PF + r + 2, ny) * nx];
            bnn[r] = FIRST ? 0.0 : bp[(size_t)clampi(jb + PF + r, 0, ny - 1) * nx];
        }
#pragma unroll
        for (int r = 0; r < PF; ++r) {
            const int j = jb + r;
            if (j < ny) {
                const double hp2 = hq[r];
                // ---- cell (j+1): Laplacian and nonlinear functions
                const double hL = __shfl_up_sync(FULL, hp1, 1), hR = __shfl_down_sync(FULL, hp1, 1);
                Lp = fma((hL + hR) - 2.0 * hp1, P.rdx2, ((hp2 + h0) - 2.0 * hp1) * P.rdy2);
                cp = cell_functions<N, M>(hp1, P);
                // ---- face j+1/2 along y
                const bool yface = (j >= 0) && (j <= ny - 2);
                const double dh = hp1 - h0;
                const double sf0 = c0.f0 + cp.f0, sf1 = c0.f1 + cp.f1;
                Face fp = face_partials(hm1, hp2, dh, sf0, sf1, c0, cp, DY);
                double phip = DY.cb * fma(sf0, Lp - L0, sf1 * dh);
                if (j == 0) fp.p1 -= fp.A;                   // ghost h(-1) == h(0): fold dF/dh_{-1}
                if (j == ny - 2) fp.p2 += fp.A;              // ghost h(ny) == h(ny-1)
                if (!yface) { fp.A = 0.0; fp.p1 = 0.0; fp.p2 = 0.0; phip = 0.0; }
                if (j >= 0) {
                    // ---- x faces of row j: i+1/2 here, i-1/2 from the left lane
                    const double f0R = __shfl_down_sync(FULL, c0.f0, 1), f1R = __shfl_down_sync(FULL, c0.f1, 1);
                    const double LR = __shfl_down_sync(FULL, L0, 1);
                    double phixp = DX.cb * fma(c0.f0 + f0R, LR - L0, (c0.f1 + f1R) * (hR0 - h0));
                    if (!xface) phixp = 0.0;
                    const double phixm = __shfl_up_sync(FULL, phixp, 1);
                    const double sD = (phixp - phixm) + (phip - phim);
                    double R;
                    if (FIRST) {
                        const double b = h0 - sD;
                        if (outl) bn[(size_t)j * nx + i] = b;
                        R = (b - h0) - sD;
                    } else {
                        R = (bq[r] - h0) - sD;
                    }
                    // ---- row j of I + s J_y:  e, c, q, a, b on rows j-2..j+2
                    const double e = fm.A, b2 = fp.A;
                    const double c = -fp.A - fm.p1;
                    const double q = 1.0 + fp.p1 - fm.p2;
                    const double a = fp.p2 - fm.A;
                    double va, vb, vz;
                    elim_row(S, e, c, q, a, b2, R, va, vb, vz);
                    if (outl) {
                        const size_t o = (size_t)j * nx + i;
                        al[o] = va; be[o] = vb; zz[o] = vz;
                    }
                }
                // ---- roll the window
                hm1 = h0; h0 = hp1; hp1 = hp2; hR0 = hR;
                c0 = cp; L0 = Lp; fm = fp; phim = phip;
            }
        }
#pragma unroll
        for (int r = 0; r < PF; ++r) { hq[r] = hn[r]; bq[r] = bnn[r]; }
    }
}

// ---------------------------------------------------------------------------------------------
// y backward:  w_j = z_j - alpha_j w_{j+1} - beta_j w_{j+2},  j = ny-1..0   (U a = b)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32)
ybwd_kernel(int nx, int ny, const double* __restrict__ al, const double* __restrict__ be,
            const double* __restrict__ zz, double* __restrict__ w)
{
    const int i = blockIdx.x * 32 + threadIdx.x;
    if (i >= nx) return;
    double w1 = 0.0, w2 = 0.0;
    for (int jt = ny - 1; jt >= 0; jt -= PF) {
        double A[PF], B[PF], Z[PF];
#pragma unroll
        for (int r = 0; r < PF; ++r) {
            const size_t o = (size_t)clampi(jt - r, 0, ny - 1) * nx + i;
            A[r] = al[o]; B[r] = be[o]; Z[r] = zz[o];
        }
#pragma unroll
        for (int r = 0; r < PF; ++r) {
            const int j = jt - r;
            if (j >= 0) {
                const double x = fma(-A[r], w1, fma(-B[r], w2, Z[r]));
                w[(size_t)j * nx + i] = x;
                w2 = w1; w1 = x;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// x forward.  A warp owns 32 rows (lane = row) and marches i = 0..nx-1 through 32x32 tiles that are
// loaded coalesced (lanes along i) into padded shared memory and read transposed (lane = row).
// Only x-neighbours are needed, so there is no halo.  Output transposed [i][j].
// ---------------------------------------------------------------------------------------------
constexpr int XT = 32;          // tile edge
constexpr int XTP = XT + 1;     // padded row length (doubles)

template <int N, int M>
__global__ void __launch_bounds__(32)
xfwd_kernel(Params P, Dir DX, const double* __restrict__ u, const double* __restrict__ w,
            double* __restrict__ alT, double* __restrict__ beT, double* __restrict__ zzT)
{
    __shared__ double sU[XT * XTP], sW[XT * XTP];
    const int nx = P.nx, ny = P.ny;
    const int lane = threadIdx.x;
    const int j0 = blockIdx.x * XT;
    const int j = j0 + lane;
    const bool rowok = j < ny;

    auto load_tile = [&](int t) {
        const int col = t * XT + lane;
        const int cc = col < nx ? col : nx - 1;
#pragma unroll 8
        for (int rr = 0; rr < XT; ++rr) {
            const int jr = (j0 + rr < ny) ? j0 + rr : ny - 1;
            sU[rr * XTP + lane] = u[(size_t)jr * nx + cc];
            sW[rr * XTP + lane] = w[(size_t)jr * nx + cc];
        }
    };
    load_tile(0);
    __syncwarp();
    // window before step i = -1:  h(-2) = h[1], h(-1) = h[0], h(0) = h[0]
    double hm1 = sU[lane * XTP + 1], h0 = sU[lane * XTP + 0], hp1 = h0;
    double wd1 = sW[lane * XTP + 0], wd0 = 0.0;            // w(i+1), w(i)
    double hlast1 = 0.0, hlast2 = 0.0;                     // h[nx-1], h[nx-2] for the right ghosts
    Cell c0 = {0, 0, 0, 0}, cp;
    Face fm = {0, 0, 0};
    Elim S = {0, 0, 0, 0, 0, 0};
    // step i consumes stream column c = i + 2 (h(i+2), w(i+2)); c runs 1 .. nx+1
    for (int i = -1; i < nx; ++i) {
        const int c = i + 2;
        double hp2, wnew = 0.0;
        if (c < nx) {
            if ((c % XT) == 0) { __syncwarp(); load_tile(c / XT); __syncwarp(); }
            hp2 = sU[lane * XTP + (c % XT)];
            wnew = sW[lane * XTP + (c % XT)];
            hlast2 = hlast1; hlast1 = hp2;
        } else {
            hp2 = (c == nx) ? hlast1 : hlast2;
        }
        cp = cell_functions<N, M>(hp1, P);
        const bool face = (i >= 0) && (i <= nx - 2);
        const double dh = hp1 - h0;
        const double sf0 = c0.f0 + cp.f0, sf1 = c0.f1 + cp.f1;
        Face fp = face_partials(hm1, hp2, dh, sf0, sf1, c0, cp, DX);
        if (i == 0) fp.p1 -= fp.A;
        if (i == nx - 2) fp.p2 += fp.A;
        if (!face) { fp.A = 0.0; fp.p1 = 0.0; fp.p2 = 0.0; }
        if (i >= 0) {
            const double e = fm.A, b2 = fp.A;
            const double cc = -fp.A - fm.p1;
            const double q = 1.0 + fp.p1 - fm.p2;
            const double a = fp.p2 - fm.A;
            double va, vb, vz;
            elim_row(S, e, cc, q, a, b2, wd0, va, vb, vz);
            if (rowok) {
                const size_t o = (size_t)i * ny + j;
                alT[o] = va; beT[o] = vb; zzT[o] = vz;
            }
        }
        hm1 = h0; h0 = hp1; hp1 = hp2;
        c0 = cp; fm = fp;
        wd0 = wd1; wd1 = wnew;
    }
}

// ---------------------------------------------------------------------------------------------
// x backward + update + residual:  v_i = z_i - alpha_i v_{i+1} - beta_i v_{i+2};  u_{k+1} = u_k + v;
// res = max |v/u_k| (2.22); also flags a non-finite or non-positive new iterate.
// `red[0]` = residual (max, as ordered bits), `red[1]` = bad-iterate flag.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32)
xbwd_kernel(int nx, int ny, const double* __restrict__ alT, const double* __restrict__ beT,
            const double* __restrict__ zzT, const double* uk, double* unew,   // uk may alias unew (in place)
            double* __restrict__ red)
{
    __shared__ double sU[XT * XTP];
    const int lane = threadIdx.x;
    const int j0 = blockIdx.x * XT;
    const int j = j0 + lane;
    const bool rowok = j < ny;
    const int jc = rowok ? j : ny - 1;
    double v1 = 0.0, v2 = 0.0, res = 0.0;
    int bad = 0;
    const int ntile = (nx + XT - 1) / XT;
    for (int t = ntile - 1; t >= 0; --t) {
        const int col = t * XT + lane;
        const int cc = col < nx ? col : nx - 1;
        __syncwarp();
#pragma unroll 8
        for (int rr = 0; rr < XT; ++rr) {
            const int jr = (j0 + rr < ny) ? j0 + rr : ny - 1;
            sU[rr * XTP + lane] = uk[(size_t)jr * nx + cc];
        }
        __syncwarp();
        const int ihi = min(nx, (t + 1) * XT) - 1;
        for (int ib = ihi; ib >= t * XT; ib -= PF) {
            double A[PF], B[PF], Z[PF];
#pragma unroll
            for (int r = 0; r < PF; ++r) {
                const size_t o = (size_t)max(ib - r, t * XT) * ny + jc;
                A[r] = alT[o]; B[r] = beT[o]; Z[r] = zzT[o];
            }
#pragma unroll
            for (int r = 0; r < PF; ++r) {
                const int i = ib - r;
                if (i >= t * XT) {
                    const double v = fma(-A[r], v1, fma(-B[r], v2, Z[r]));
                    const double uo = sU[lane * XTP + (i - t * XT)];
                    const double un = uo + v;
                    const double rr = fabs(v / uo);
                    if (rowok) {
                        if (!(rr <= res)) res = rr;          // NaN sticks
                        if (!(un > 0.0) || isinf(un)) bad = 1;
                    }
                    sU[lane * XTP + (i - t * XT)] = un;
                    v2 = v1; v1 = v;
                }
            }
        }
        __syncwarp();
        if (col < nx) {
#pragma unroll 8
            for (int rr = 0; rr < XT; ++rr)
                if (j0 + rr < ny) unew[(size_t)(j0 + rr) * nx + col] = sU[rr * XTP + lane];
        }
    }
    if (res != res) res = __longlong_as_double(0x7ff8000000000000LL);   // canonical +NaN for the bit-max
    res = warp_max_nonneg(res);
    bad = __any_sync(0xffffffffu, bad);
    if (lane == 0) {
        atomic_max_nonneg(red, res);
        if (bad) atomic_max_nonneg(red + 1, 1.0);
    }
}

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
