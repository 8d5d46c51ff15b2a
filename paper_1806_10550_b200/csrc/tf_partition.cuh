// tf_partition.cuh -- intra-line parallel variant of the isolated pentadiagonal solver.
//
// The paper solves one system per thread and names "the SPIKE method or cyclical reduction" as the way to
// parallelise a single system.  Thread-per-line needs >= ~20 000 lines to fill a B200; with
// few long lines (nsys/32 marching warps) the serial chain len x 52 cycles is all there is.  This variant cuts
// every line into P chunks and runs three steps (a partition / SPIKE-type reduced-interface scheme):
//   1. interface pass   per (line, chunk): eliminate the chunk's rows downwards AND upwards, each march carrying
//                       three right-hand sides -- rhs and the two columns that couple the chunk to the two
//                       unknowns just outside its far end.  The last two rows of a march are exact relations
//                       between the chunk's two end unknowns and the four unknowns outside it
//                       (penta_col_iface_kernel / penta_row_iface_kernel, nothing else is stored);
//   2. reduced system   per line: the 4P end unknowns (t_p = first two, b_p = last two of chunk p) satisfy a
//                       block-bidiagonal-coupled system with 2x2 blocks; solved serially (penta_reduced_kernel);
//   3. chunk solves     every chunk is now an independent pentadiagonal system whose first/last two right-hand
//                       sides are corrected by the known outside values: the two-sided TMA kernels of the LU
//                       variant run on all chunks at once (blockIdx.z = chunk).
// Same solution as the LU of PAPER.md:729-734 up to rounding (no pivoting in either; the reduced system of a
// diagonally dominant matrix is diagonally dominant).  Traffic per unknown: 2 x 48 B (step 1) + 104 B (step 3).
#pragma once
#include "tf_device.cuh"
#include "tf_tma.cuh"
#include "tf_async.cuh"

namespace tf {

// chunk p of P covers rows [chunk_lo(p), chunk_lo(p+1)) of a line of N; interior bounds are multiples of 16
// (the tile width of the row-direction kernels, so that no two CTAs ever store into the same tile)
__host__ __device__ __forceinline__ int chunk_lo(int p, int P, int N)
{
    return p <= 0 ? 0 : (p >= P ? N : (int)(((long long)p * N / P) / 16 * 16));
}
__host__ __device__ __forceinline__ int chunk_mid(int lo, int hi) { return lo + ((hi - lo) / 2) / 16 * 16; }

constexpr int IF_VALS = 10;      // per (chunk, march): alpha, beta, z_rhs, z_far, z_near of the last and the last-but-one row
constexpr int RC_VALS = 12;      // per chunk: ht(2), Ct(4), hb(2), Cb(4) of the reduced elimination

// one more right-hand side carried through elim2_row's elimination (numerator of the unfinished row, z of row i-2)
struct Elim2R { double s1, z2; };

// elim2_row (tf_device.cuh) with two extra right-hand sides yf, yn; emits the final coefficients of row i-1
__device__ __forceinline__ void elim2_row3(Elim2& S, Elim2R& F, Elim2R& G, double e, double c, double q, double a, double b,
                                           double y, double yf, double yn)
{
    const double gam = fma(-S.a2, e, c);
    const double T = fma(-S.b2, e, q);
    const double g = S.p1 * gam;
    const double bg = S.b1 * gam;
    const double sy = fma(-S.z2, e, y);
    const double syf = fma(-F.z2, e, yf);
    const double syn = fma(-G.z2, e, yn);
    const double u1 = fma(-g, S.y1, T);
    const double Gg = g * S.y1;
    const double mu = fma(-Gg, S.t1, u1);
    double y0;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(mu));
    const double ee = fma(-mu, y0, 1.0);
    const double tt = fma(ee, ee, ee);
    const double r1 = fma(S.y1, S.t1, S.y1);
    const double al = S.p1 * r1, be = S.b1 * r1, zz = S.s1 * r1, zf = F.s1 * r1, zn = G.s1 * r1;
    const double p = fma(-bg, r1, a);
    S.s1 = fma(-zz, gam, sy);
    F.s1 = fma(-zf, gam, syf);
    G.s1 = fma(-zn, gam, syn);
    S.a2 = al; S.b2 = be; S.z2 = zz; F.z2 = zf; G.z2 = zn;
    S.y1 = y0; S.t1 = tt; S.p1 = p; S.b1 = b;
}

// after the last row of a march: write the ten interface values (lanes along the systems, stride nsys)
__device__ __forceinline__ void iface_emit(const Elim2& S, const Elim2R& F, const Elim2R& G, double* out, size_t nsys, int ok)
{
    const double r1 = fma(S.y1, S.t1, S.y1);
    if (ok) {
        out[0] = S.p1 * r1; out[nsys] = S.b1 * r1; out[2 * nsys] = S.s1 * r1; out[3 * nsys] = F.s1 * r1; out[4 * nsys] = G.s1 * r1;
        out[5 * nsys] = S.a2; out[6 * nsys] = S.b2; out[7 * nsys] = S.z2; out[8 * nsys] = F.z2; out[9 * nsys] = G.z2;
    }
}

struct Maps6 { CUtensorMap m[6]; };      // e, c, d, a, b, rhs

// ---- step 1, systems = columns (lanes along the contiguous index).  grid (ceil(ncol/32), 2, P): blockIdx.y = march
// (0: rows lo .. hi-1 downwards, 1: rows hi-1 .. lo upwards as the reversed system e<->b, c<->a), blockIdx.z = chunk.
// The far / near outside unknowns of a march are the two just before its first row: x_{lo-2}, x_{lo-1} (down) or
// x_{hi+1}, x_{hi} (up); their columns are (e_0, 0, ..) and (c_0, e_1, 0, ..) in the march's own orientation.
// out: [P][2][IF_VALS][ncol].
template <int NST, int RS>
__global__ void __launch_bounds__(32)
penta_col_iface_kernel(const __grid_constant__ Maps6 M, int nrow, int ncol, int P, double* __restrict__ out,
                       int Pg, int p_off)
{
    extern __shared__ unsigned char raw[];
    unsigned char* base = align1024(raw);
    constexpr int BOX = RS * 32;
    double* sm = reinterpret_cast<double*>(base);            // [NST][6][RS][32]
    uint64_t* full = reinterpret_cast<uint64_t*>(base + (size_t)NST * 6 * BOX * 8);
    const int lane = threadIdx.x;
    const int i0 = blockIdx.x * 32, i = i0 + lane;
    const int dir = blockIdx.y, p = blockIdx.z;
    const int lo = chunk_lo(p, P, nrow), hi = chunk_lo(p + 1, P, nrow);
    const int ntile = (hi - lo + RS - 1) / RS;
    // Pg, p_off: the arrays may be one slab of a line that continues on other devices (tf_penta_slab_*): local chunk p
    // is chunk p_off + p of Pg.  Single device: Pg = P, p_off = 0.
    const bool outside = dir ? (p_off + p < Pg - 1) : (p_off + p > 0);   // does this march have outside unknowns at its start?
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
    Elim2R F = {0.0, 0.0}, G = {0.0, 0.0};
    const int oe = dir ? 4 * BOX : 0, oc = dir ? 3 * BOX : BOX, oa = dir ? BOX : 3 * BOX, ob = dir ? 0 : 4 * BOX;
    int k = 0;                                               // rows eliminated so far
    for (int q = 0; q < ntile; ++q) {
        const int s = q % NST;
        mbar_wait(full + s, (q / NST) & 1);
        const int jb = box_row(q);
        const double* d = sm + (size_t)s * 6 * BOX + lane;
        if (jb >= lo && jb + RS <= hi && q > 0) {
#pragma unroll
            for (int rr = 0; rr < RS; ++rr) {
                const int r = dir ? RS - 1 - rr : rr;
                elim2_row3(S, F, G, d[oe + r * 32], d[oc + r * 32], d[2 * BOX + r * 32], d[oa + r * 32], d[ob + r * 32],
                           d[5 * BOX + r * 32], 0.0, 0.0);
            }
            k += RS;
        } else {
            for (int rr = 0; rr < RS; ++rr) {
                const int r = dir ? RS - 1 - rr : rr;
                const int j = jb + r;
                if (j >= lo && j < hi) {
                    const double e = d[oe + r * 32], c = d[oc + r * 32];
                    const double yf = (outside && k == 0) ? e : 0.0;
                    const double yn = outside ? (k == 0 ? c : (k == 1 ? e : 0.0)) : 0.0;
                    elim2_row3(S, F, G, e, c, d[2 * BOX + r * 32], d[oa + r * 32], d[ob + r * 32], d[5 * BOX + r * 32], yf, yn);
                    ++k;
                }
            }
        }
        __syncwarp();
        issue(q + NST);
    }
    iface_emit(S, F, G, out + ((size_t)(p * 2 + dir) * IF_VALS) * ncol + i, (size_t)ncol, i < ncol);
}

// ---- step 1, systems = rows (contiguous).  lane <-> row of a block of 32 rows; [32 rows x 16 cols] TMA boxes with the
// 128-byte swizzle as in penta_row_fwd2_kernel.  grid (ceil(nrow/32), 2, P).  out: [P][2][IF_VALS][nrow].
template <int NST>
__global__ void __launch_bounds__(32)
penta_row_iface_kernel(const __grid_constant__ Maps6 M, int nrow, int ncol, int P, double* __restrict__ out,
                       int Pg, int p_off)
{
    constexpr int CS = 16;
    constexpr int TILE = 32 * CS * 8;
    extern __shared__ unsigned char raw[];
    unsigned char* base = align1024(raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(base + (size_t)NST * 6 * TILE);
    const int lane = threadIdx.x;
    const int r0 = blockIdx.x * 32;
    const int dir = blockIdx.y, p = blockIdx.z;
    const int lo = chunk_lo(p, P, ncol), hi = chunk_lo(p + 1, P, ncol);
    const int ntile = (hi - lo + CS - 1) / CS;
    const bool outside = dir ? (p_off + p < Pg - 1) : (p_off + p > 0);
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
    Elim2R F = {0.0, 0.0}, G = {0.0, 0.0};
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
        if (ib >= lo && ib + CS <= hi && q > 0) {
#pragma unroll
            for (int cc = 0; cc < CS; ++cc) {
                const int c = dir ? CS - 1 - cc : cc;
                elim2_row3(S, F, G, at(oe, c), at(oc, c), at(2 * TILE, c), at(oa, c), at(ob, c), at(5 * TILE, c), 0.0, 0.0);
            }
            k += CS;
        } else {
            for (int cc = 0; cc < CS; ++cc) {
                const int c = dir ? CS - 1 - cc : cc;
                const int i = ib + c;
                if (i >= lo && i < hi) {
                    const double e = at(oe, c), cv = at(oc, c);
                    const double yf = (outside && k == 0) ? e : 0.0;
                    const double yn = outside ? (k == 0 ? cv : (k == 1 ? e : 0.0)) : 0.0;
                    elim2_row3(S, F, G, e, cv, at(2 * TILE, c), at(oa, c), at(ob, c), at(5 * TILE, c), yf, yn);
                    ++k;
                }
            }
        }
        __syncwarp();
        issue(q + NST);
    }
    iface_emit(S, F, G, out + ((size_t)(p * 2 + dir) * IF_VALS) * nrow + r0 + lane, (size_t)nrow, r0 + lane < nrow);
}

// ---- step 2: the reduced system, one thread per line.  With t_p = (x_lo, x_lo+1), b_p = (x_hi-2, x_hi-1) of chunk p,
// the last two rows of the two marches read (after removing the in-chunk coupling of the last-but-one row)
//     t_p + Lt_p b_{p-1} + Ut_p t_{p+1} = gt_p,      b_p + Lb_p b_{p-1} + Ub_p t_{p+1} = gb_p        (2x2 blocks).
// Forward: b_{p-1} = hb_{p-1} - Cb_{p-1} t_p  =>  (I - Lt_p Cb_{p-1}) t_p = gt_p - Lt_p hb_{p-1} - Ut_p t_{p+1}, i.e.
// t_p = ht_p - Ct_p t_{p+1}, and b_p = hb_p - Cb_p t_{p+1} with hb_p = gb_p - Lb_p hb_{p-1} + (Lb_p Cb_{p-1}) ht_p,
// Cb_p = Ub_p + (Lb_p Cb_{p-1}) Ct_p.  Backward from t_P = 0.  iface: [P][2][IF_VALS][nsys]; rc: [P][RC_VALS][nsys]
// scratch; X: [P][4][nsys] = (t_p, b_p).  Coefficients that multiply unknowns outside the line (first chunk's upward
// march, last chunk's downward march) are formed from ignored band entries and are dropped by selection.
__global__ void __launch_bounds__(32)
penta_reduced_kernel(int nsys, int P, const double* __restrict__ iface, double* __restrict__ rc, double* __restrict__ X)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nsys) return;
    const size_t n = (size_t)nsys;
    double hb0 = 0.0, hb1 = 0.0, cb00 = 0.0, cb01 = 0.0, cb10 = 0.0, cb11 = 0.0;
    // The loop is a short dependent chain (~0.1 us per chunk) fed by 20 loads per chunk: a cp.async ring keeps the
    // values of the next RD chunks in flight (loading them where they are used cost a full memory latency per
    // chunk: 48 us for 37 chunks; one chunk of register prefetch: 34 us).  Every thread copies and reads its own
    // slots, so cp.async.wait_group is the only synchronisation.
    constexpr int RD = 8;
    __shared__ double ring[RD][2 * IF_VALS][32];
    const int lane = threadIdx.x;
    auto fetch = [&](int q) {
        if (q < P) {
            const double* src = iface + (size_t)q * 2 * IF_VALS * n + i;
#pragma unroll
            for (int k = 0; k < 2 * IF_VALS; ++k) cp_async8(&ring[q % RD][k][lane], src + (size_t)k * n);
        }
        cp_async_commit();
    };
#pragma unroll
    for (int q = 0; q < RD; ++q) fetch(q);
    double v[2 * IF_VALS];
    for (int p = 0; p < P; ++p) {
        cp_async_wait<RD - 1>();
#pragma unroll
        for (int k = 0; k < 2 * IF_VALS; ++k) v[k] = ring[p % RD][k][lane];
        __syncwarp();
        fetch(p + RD);
        // downward march: row hi-1 (0..4), hi-2 (5..9); upward march: row lo (10..14), lo+1 (15..19)
        const double d1a = v[0], d1b = v[1], d1y = v[2], d1f = v[3], d1n = v[4];
        const double d2a = v[5], d2b = v[6], d2y = v[7], d2f = v[8], d2n = v[9];
        const double u1a = v[10], u1b = v[11], u1y = v[12], u1f = v[13], u1n = v[14];
        const double u2a = v[15], u2b = v[16], u2y = v[17], u2f = v[18], u2n = v[19];
        const bool first = p == 0, last = p == P - 1;
        const double gt0 = u1y, gt1 = fma(-u2a, u1y, u2y);
        const double gb1 = d1y, gb0 = fma(-d2a, d1y, d2y);
        const double lt00 = first ? 0.0 : u1b, lt01 = first ? 0.0 : u1a;
        const double lt10 = first ? 0.0 : -u2a * u1b, lt11 = first ? 0.0 : fma(-u2a, u1a, u2b);
        const double lb00 = first ? 0.0 : fma(-d2a, d1f, d2f), lb01 = first ? 0.0 : fma(-d2a, d1n, d2n);
        const double lb10 = first ? 0.0 : d1f, lb11 = first ? 0.0 : d1n;
        const double ut00 = last ? 0.0 : u1n, ut01 = last ? 0.0 : u1f;
        const double ut10 = last ? 0.0 : fma(-u2a, u1n, u2n), ut11 = last ? 0.0 : fma(-u2a, u1f, u2f);
        const double ub00 = last ? 0.0 : fma(-d2a, d1a, d2b), ub01 = last ? 0.0 : -d2a * d1b;
        const double ub10 = last ? 0.0 : d1a, ub11 = last ? 0.0 : d1b;
        // M = I - Lt Cb_prev
        const double m00 = 1.0 - (lt00 * cb00 + lt01 * cb10), m01 = -(lt00 * cb01 + lt01 * cb11);
        const double m10 = -(lt10 * cb00 + lt11 * cb10), m11 = 1.0 - (lt10 * cb01 + lt11 * cb11);
        const double rdet = 1.0 / (m00 * m11 - m01 * m10);
        const double i00 = m11 * rdet, i01 = -m01 * rdet, i10 = -m10 * rdet, i11 = m00 * rdet;
        const double r0 = gt0 - (lt00 * hb0 + lt01 * hb1), r1 = gt1 - (lt10 * hb0 + lt11 * hb1);
        const double ht0 = i00 * r0 + i01 * r1, ht1 = i10 * r0 + i11 * r1;
        const double ct00 = i00 * ut00 + i01 * ut10, ct01 = i00 * ut01 + i01 * ut11;
        const double ct10 = i10 * ut00 + i11 * ut10, ct11 = i10 * ut01 + i11 * ut11;
        // K = Lb Cb_prev
        const double k00 = lb00 * cb00 + lb01 * cb10, k01 = lb00 * cb01 + lb01 * cb11;
        const double k10 = lb10 * cb00 + lb11 * cb10, k11 = lb10 * cb01 + lb11 * cb11;
        const double nhb0 = gb0 - (lb00 * hb0 + lb01 * hb1) + (k00 * ht0 + k01 * ht1);
        const double nhb1 = gb1 - (lb10 * hb0 + lb11 * hb1) + (k10 * ht0 + k11 * ht1);
        cb00 = ub00 + (k00 * ct00 + k01 * ct10); cb01 = ub01 + (k00 * ct01 + k01 * ct11);
        cb10 = ub10 + (k10 * ct00 + k11 * ct10); cb11 = ub11 + (k10 * ct01 + k11 * ct11);
        hb0 = nhb0; hb1 = nhb1;
        double* R = rc + (size_t)p * RC_VALS * n + i;
        R[0] = ht0; R[n] = ht1; R[2 * n] = ct00; R[3 * n] = ct01; R[4 * n] = ct10; R[5 * n] = ct11;
        R[6 * n] = hb0; R[7 * n] = hb1; R[8 * n] = cb00; R[9 * n] = cb01; R[10 * n] = cb10; R[11 * n] = cb11;
    }
    double t0 = 0.0, t1 = 0.0;                                // t_{p+1}
    cp_async_wait<0>();
    auto fetch_rc = [&](int q) {                                // q-th chunk from the end
        if (q < P) {
            const double* src = rc + (size_t)(P - 1 - q) * RC_VALS * n + i;
#pragma unroll
            for (int k = 0; k < RC_VALS; ++k) cp_async8(&ring[q % RD][k][lane], src + (size_t)k * n);
        }
        cp_async_commit();
    };
#pragma unroll
    for (int q = 0; q < RD; ++q) fetch_rc(q);
    double w[RC_VALS];
    for (int p = P - 1; p >= 0; --p) {
        const int q = P - 1 - p;
        cp_async_wait<RD - 1>();
#pragma unroll
        for (int k = 0; k < RC_VALS; ++k) w[k] = ring[q % RD][k][lane];
        __syncwarp();
        fetch_rc(q + RD);
        const double nt0 = w[0] - (w[2] * t0 + w[3] * t1), nt1 = w[1] - (w[4] * t0 + w[5] * t1);
        const double b0 = w[6] - (w[8] * t0 + w[9] * t1), b1 = w[7] - (w[10] * t0 + w[11] * t1);
        double* x = X + (size_t)p * 4 * n + i;
        x[0] = nt0; x[n] = nt1; x[2 * n] = b0; x[3 * n] = b1;
        t0 = nt0; t1 = nt1;
    }
}

}  // namespace tf
