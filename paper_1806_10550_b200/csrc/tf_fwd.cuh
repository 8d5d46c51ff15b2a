// tf_fwd.cuh -- warp-specialised forward kernels (assembly + LU forward elimination), S1-S6 forward halves.
//
// Why: a sweep has only nx (ny) independent lines = 256 warps at 8192^2 for 592 SM sub-partitions, and the
// assembly of one matrix row costs ~55 fp64 instructions against 17 for the elimination recurrence, which is
// a serial chain (52 cycles per row).  If the thread that carries the recurrence also assembles, most fp64
// pipes idle.  So the work of a strip of lines is split:
//   * NP producer warps assemble rows (bands A,c,q,a and right-hand side R) for disjoint chunks --
//     embarrassingly parallel -- and hand them over through a shared-memory ring;
//   * 1 consumer warp runs the pentadiagonal recurrence and streams alpha,beta,z out;
//   * every line is eliminated from both ends by two such teams (two-sided / twisted factorisation), and one
//     CTA per SM hosts four teams, one per SM sub-partition.
// Hand-over is by mbarriers (full/empty per slot), no __syncthreads in the steady state.
// has the measurements behind each of these choices (register reallocation between the consumer and producer
// warpgroups with setmaxnreg was also measured: no gain).
#pragma once
#include "tf_device.cuh"
#include "tf_tma.cuh"
#include <type_traits>

namespace tf {

#ifndef TF_ROTATE_Y
#define TF_ROTATE_Y 1
#endif
// What bounds these kernels was measured with timing-only probe builds (one ingredient left out or added at a time);
// the results are in profiles/r02_ncu.md, the switches are gone from the source.
constexpr int YW_VALID = 28;     // columns per strip (lanes 2..29; lanes 0,1,30,31 are x-halo)

// Warps of a forward CTA.  With one team per CTA (NSUB = 1, small grids) the consumer keeps SM sub-partition 0 to itself:
// warps 4, 8, ... (which would share it) are launched idle, the producers are the warps with warp % 4 != 0.
#ifndef TF_N1_SKIP0
#define TF_N1_SKIP0 1
#endif
#ifndef TF_N2_SKIP0
#define TF_N2_SKIP0 0
#endif
// the same for two teams per CTA (both consumers on sub-partition 0, warps 0 and 4) was measured slower (4096^2: y forward
// 0.155 -> 0.163 ms, x forward 0.152 -> 0.167 ms) and is off
__host__ __device__ constexpr bool fwd_sp0(int nsub) { return (nsub == 1 && TF_N1_SKIP0) || (nsub == 2 && TF_N2_SKIP0); }
__host__ __device__ constexpr int fwd_warps(int nsub, int np)
{
    if (!fwd_sp0(nsub)) return nsub * (np + 1);
    int w = 4 * (nsub - 1) + 1;                       // the last consumer warp
    while (w - (w + 3) / 4 < nsub * np) ++w;           // warps 0 .. w-1 hold w - ceil(w/4) producers
    return w;
}

// rolling state of a thread marching down a column
struct YState {
    double hm1, h0, hp1;         // h(j-1), h(j), h(j+1)
    double hR0;                  // h(j)[i+1]
    Cell c0;                     // cell (j)
    double L0;                   // lap h (j)
    Face fm;                     // face j-1/2 (folded / zeroed)
    double phim;                 // s*Fy(j-1/2)/dy
};

// MODE 0: bring in cell (j+1) only;  1: also face j+1/2;  2: also produce row j (bands + R).
// out6 = {A_{j+1/2}, c, q, a, R, A_{j-1/2}}
// INTERIOR: all faces touched are interior and unfolded (1 <= j <= ny-3): no boundary logic at all.
template <int N, int M, int MODE, bool INTERIOR>
__device__ __forceinline__ void y_advance(YState& S, int j, double hp2, const Params& P, const Dir& DX, const Dir& DY,
                                          bool xface, double rhs_in, double* out6, double& sD_out)
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
        out6[0] = fp.A;
        out6[1] = -fp.A - S.fm.p1;
        out6[2] = 1.0 + fp.p1 - S.fm.p2;
        out6[3] = fp.p2 - S.fm.A;
        out6[4] = (rhs_in - S.h0) - sD;            // FIRST: caller passes rhs_in = b, fixed up below
        out6[5] = S.fm.A;
    }
    S.hm1 = S.h0; S.h0 = S.hp1; S.hp1 = hp2; S.hR0 = hR;
    S.c0 = cp; S.L0 = Lp;
    if (MODE >= 1) { S.fm = fp; S.phim = phip; }
}

// ---------------------------------------------------------------------------------------------
// y forward, two-sided ("burn at both ends", twisted factorisation): the lines of a strip are eliminated
// from row 0 downwards (half 0, rows [0, mid)) and from row ny-1 upwards (half 1, rows [mid, ny)) by two
// independent CTAs; the back-substitution kernel joins them with a 4x4 interface solve per line.  Same
// operation count as the one-sided LU of PAPER.md:729-734, half the serial chain, twice the marching
// warps (the chain x ny was the floor of the one-sided kernel).  For half 1 the system is taken in
// reversed order k = ny-1-j: e' = b, c' = a, a' = c, b' = e, so its producers hand over A_{j-1/2}
// instead of A_{j+1/2} and the consumer swaps the c and a planes; everything else is shared.
// Coefficients of half 0 mean x_j = z_j - al_j x_{j+1} - be_j x_{j+2}; of half 1: x_j = z_j - al_j x_{j-1} - be_j x_{j-2}.
//
// CTA = warp 0 (consumer: the recurrence) + NP producer warps (assembly).  The hand-over ring has NCH
// slots of ONE CHUNK (RP rows of one producer) each: chunk c is assembled by producer c % NP into slot
// c % NCH, so RP can be large (the two warm-up rows of a chunk are amortised over RP rows) while the ring
// stays small.  Inputs arrive by TMA, one box per chunk, issued a chunk ahead (see the producer loop).
// ---------------------------------------------------------------------------------------------
template <int N, int M, bool FIRST, int NP, int RP, int NCH, int NSUB>
__global__ void __launch_bounds__(32 * fwd_warps(NSUB, NP), 1)
yfwd_ws_kernel(const __grid_constant__ CUtensorMap mU, const __grid_constant__ CUtensorMap mB, int use_tma,
               Params P, Dir DX, Dir DY, int mid, const double* __restrict__ u, double* __restrict__ bn,
               double* __restrict__ al, double* __restrict__ be, double* __restrict__ zz, Gate gate)
{
    if (gate_closed(gate)) return;
    if (gate.s) { const double sdev = __ldcg(gate.s); DX = dir_of(sdev, P.dx); DY = dir_of(sdev, P.dy); }
    // One CTA per SM: NSUB = 4 sub-problems q = warp % 4 (two adjacent strips x two halves), each with its own
    // ring and its own consumer + NP producers.  Warps w, w+4, w+8, ... share an SM sub-partition, so every
    // sub-partition gets exactly one consumer and NP producers (the consumers' dependent chains and the
    // producers' fp64 work are spread evenly over the four issue ports).  Grids with at most one strip per SM
    // use NSUB = 2 (one strip x two halves per CTA) so that twice as many SMs work.
    // Shared memory: 4 rings [NCH][5][RP][32] | 4*NP input stagings [(RP+4) + RP][32] | mbarriers.
    // NCH >= NP keeps every producer less than one ring lap ahead of the consumer, which the parity waits need
    // (a waiter two phases ahead would see the wrong parity as "done"; NP = 4, NCH = 3 hangs).
    static_assert(NCH >= NP, "ring slots must not be fewer than producers");
    constexpr int SV = RP * 32;                       // doubles per value plane of a slot
    constexpr size_t RING = (size_t)NCH * 5 * SV * 8;                // bytes per sub-problem
    constexpr size_t STG = (size_t)(2 * RP + 4) * 32 * 8;            // bytes per producer: rows of u, then rows of b^n
    extern __shared__ __align__(128) unsigned char raw[];
    const int nx = P.nx, ny = P.ny;
    const int warp = uniform_warp_idx(), lane = threadIdx.x & 31;
    // role 0: consumer, 1..NP: producers.  Warp w runs on SM sub-partition w % 4: consumer q sits on sub-partition q,
    // its producers (TF_ROTATE_Y) on the sub-partitions after it, so that a team's assembly burst uses several fp64
    // pipes while the other teams' consumers (dependent chains, mostly idle issue slots) share them
    // (rotation not for the NLC cells, whose exp and extra reciprocals make the producers the fp64-heavier side: +1.5 %)
    int role, q;
    bool idle = false;
    if (fwd_sp0(NSUB)) {                              // consumers: warps 0, 4, ..; producers: the warps with warp % 4 != 0
        if (warp % 4 == 0) { role = 0; q = warp / 4; idle = warp / 4 >= NSUB; }
        else { const int p = warp - warp / 4 - 1; q = p % NSUB; role = 1 + p / NSUB; idle = role > NP; }
        if (idle) { role = 1; q = 0; }
    } else {
        role = warp / NSUB;
        q = (TF_ROTATE_Y && N != MODEL_NLC) ? (warp % NSUB + NSUB * NP - role) % NSUB : warp % NSUB;
    }
    double* sm = reinterpret_cast<double*>(raw + q * RING);          // [NCH][5][RP][32]
    uint64_t* bars = reinterpret_cast<uint64_t*>(raw + NSUB * RING + NSUB * NP * STG);
    uint64_t* full = bars + q * 2 * NCH;
    uint64_t* empty = full + NCH;
    if (role == 0 && lane == 0) {
#pragma unroll
        for (int s = 0; s < NCH; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); }
        for (int p = 0; p < NP; ++p) mbar_init(bars + 2 * NSUB * NCH + q * NP + p, 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (idle) return;
    // NSUB = 1 (grids with at most one team per SM: sides <= ~2070): one team per CTA, blockIdx.x = 2 strip + half
    constexpr int SPC = NSUB >= 2 ? NSUB / 2 : 1;     // strips per CTA
    const int strip = NSUB >= 2 ? SPC * (int)blockIdx.x + (q % SPC) : (int)blockIdx.x / 2;
    if (strip * YW_VALID >= nx) return;               // odd strip count: the last CTA has one strip
    const int i = strip * YW_VALID - 2 + lane;
    const int dir = NSUB >= 2 ? q / SPC : (int)blockIdx.x % 2;   // 0: rows 0 .. mid-1 downwards, 1: rows ny-1 .. mid upwards
    const int nrows = dir ? ny - mid : mid;           // rows of this half
    const int nchunk = (nrows + RP - 1) / RP;
    const int jmin = dir ? mid : 0, jmax = dir ? ny : mid;    // this half owns rows [jmin, jmax)
    const int outl = ((lane >= 2) && (lane < 2 + YW_VALID) && (i < nx)) ? 1 : 0;

    if (role > 0) {
        // ------------------------------------------------------------------ producer pw: chunks pw, pw+NP, ...
        const int pw = role - 1;
        const int ic = ghost(i, nx);
        const bool xface = (i >= 0) && (i <= nx - 2);
        const double* up = u + ic;
        const double* bp = bn + ic;
        // Input staging: one TMA box of RP+4 rows of u and one of RP rows of b^n per interior chunk, issued one
        // chunk ahead (right after the previous chunk's rows were copied to registers), so that the chunk's
        // global-memory latency overlaps the assembly of the chunk before it.  Boundary chunks, and grids whose
        // row pitch is not a multiple of 16 bytes, load directly.
        double* stg = reinterpret_cast<double*>(raw + NSUB * RING + (size_t)(q * NP + pw) * STG);
        uint64_t* sbar = bars + 2 * NSUB * NCH + q * NP + pw;
        const int col0 = strip * YW_VALID - 2;
        const int srcl = lane + (ic - i);                      // lane holding my ghost column (edge strips)
        const bool edge = (col0 < 0) || (col0 + 32 > nx);
        auto chunk_lo = [&](int c) { return dir ? ny - (c + 1) * RP : c * RP; };
        auto is_interior = [&](int jlo) { return (jlo >= 2) && (jlo + RP + 1 <= ny - 2) && (jlo >= jmin) && (jlo + RP <= jmax); };
        auto issue_tma = [&](int c) {
            if (use_tma && c < nchunk && lane == 0) {
                const int jl = chunk_lo(c);
                if (is_interior(jl)) {
                    mbar_expect_tx(sbar, (uint32_t)((FIRST ? RP + 4 : 2 * RP + 4) * 32 * 8));
                    tma_load_2d(stg, &mU, col0, jl - 2, sbar);
                    if (!FIRST) tma_load_2d(stg + (RP + 4) * 32, &mB, col0, jl, sbar);
                }
            }
        };
        issue_tma(pw);
        unsigned ntma = 0;                                      // boxes consumed so far (staging barrier phase)
        for (int c = pw; c < nchunk; c += NP) {
            const int s = c % NCH;
            const int jlo = chunk_lo(c);                        // the chunk is rows jlo .. jlo+RP-1
            const bool interior = is_interior(jlo);
            double hq[RP + 4], bq[RP];
            if (interior && use_tma) {
                mbar_wait(sbar, ntma & 1);
                ++ntma;
#pragma unroll
                for (int k = 0; k < RP + 4; ++k) hq[k] = stg[k * 32 + lane];
#pragma unroll
                for (int k = 0; k < RP; ++k) bq[k] = FIRST ? 0.0 : stg[(RP + 4 + k) * 32 + lane];
                if (edge) {                                     // reflect the ghost columns (TMA zero-fills them)
#pragma unroll
                    for (int k = 0; k < RP + 4; ++k) hq[k] = __shfl_sync(0xffffffffu, hq[k], srcl);
                }
            } else if (interior) {
                const double* hp = up + (size_t)(jlo - 2) * nx;
#pragma unroll
                for (int k = 0; k < RP + 4; ++k) hq[k] = hp[(size_t)k * nx];
                const double* bq0 = bp + (size_t)jlo * nx;
#pragma unroll
                for (int k = 0; k < RP; ++k) bq[k] = FIRST ? 0.0 : bq0[(size_t)k * nx];
            } else {
#pragma unroll
                for (int k = 0; k < RP + 4; ++k) hq[k] = up[(size_t)ghost(jlo - 2 + k, ny) * nx];
#pragma unroll
                for (int k = 0; k < RP; ++k) bq[k] = FIRST ? 0.0 : bp[(size_t)clampi(jlo + k, 0, ny - 1) * nx];
            }
            __syncwarp();
            issue_tma(c + NP);                                  // staging is free again: fetch my next chunk
            mbar_wait(empty + s, ((c / NCH) & 1) ^ 1);
            // slot row of chunk row r: r (half 0), RP-1-r (half 1)
            double* st = sm + (size_t)s * 5 * SV + (dir ? RP - 1 : 0) * 32 + lane;
            const int sstep = dir ? -32 : 32;
            YState S;
            S.hm1 = 0.0; S.h0 = hq[0]; S.hp1 = hq[1]; S.hR0 = 0.0;
            S.c0 = {0, 0, 0, 0}; S.L0 = 0.0; S.fm = {0, 0, 0}; S.phim = 0.0;
            double o6[6], sD;
            if (interior) {
                y_advance<N, M, 0, true>(S, jlo - 2, hq[2], P, DX, DY, xface, 0.0, o6, sD);
                y_advance<N, M, 1, true>(S, jlo - 1, hq[3], P, DX, DY, xface, 0.0, o6, sD);
                double* bo = bn + (size_t)jlo * nx + i;
#pragma unroll
                for (int r = 0; r < RP; ++r) {
                    const double hcur = S.h0;
                    y_advance<N, M, 2, true>(S, jlo + r, hq[r + 4], P, DX, DY, xface, FIRST ? hcur : bq[r], o6, sD);
                    if (FIRST) {
                        const double b = hcur - sD;
                        st_if(outl, bo + (size_t)r * nx, b);
                        o6[4] = (b - hcur) - sD;
                    }
                    double* sr = st + r * sstep;
                    sr[0] = dir ? o6[5] : o6[0]; sr[SV] = o6[1]; sr[2 * SV] = o6[2]; sr[3 * SV] = o6[3]; sr[4 * SV] = o6[4];
                }
            } else {
                y_advance<N, M, 0, false>(S, jlo - 2, hq[2], P, DX, DY, xface, 0.0, o6, sD);
                y_advance<N, M, 1, false>(S, jlo - 1, hq[3], P, DX, DY, xface, 0.0, o6, sD);
#pragma unroll
                for (int r = 0; r < RP; ++r) {
                    const int j = jlo + r;
                    const double hcur = S.h0;
                    y_advance<N, M, 2, false>(S, j, hq[r + 4], P, DX, DY, xface, FIRST ? hcur : bq[r], o6, sD);
                    if (j >= jmin && j < jmax) {
                        if (FIRST) {
                            const double b = hcur - sD;
                            if (outl) bn[(size_t)j * nx + i] = b;
                            o6[4] = (b - hcur) - sD;
                        }
                        double* sr = st + r * sstep;
                        sr[0] = dir ? o6[5] : o6[0]; sr[SV] = o6[1]; sr[2 * SV] = o6[2]; sr[3 * SV] = o6[3]; sr[4 * SV] = o6[4];
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(full + s);
        }
    } else {
        // ------------------------------------------------------------------ consumer: the recurrence.
        // elim2_row emits the coefficients of the PREVIOUS row, so every store goes one row behind.
        Elim2 S = elim2_init();
        double e = 0.0;
        const int step = dir ? -nx : nx;
        int o = (dir ? ny : -1) * nx + i;                 // the row before the first one (32-bit element offset)
        const int offc = dir ? 3 * SV : SV, offa = dir ? SV : 3 * SV;   // half 1: c' = a, a' = c
        for (int c = 0; c < nchunk; ++c) {
            const int s = c % NCH;
            mbar_wait(full + s, (c / NCH) & 1);
            const double* st = sm + (size_t)s * 5 * SV + lane;
            const double* stc = st + offc;
            const double* sta = st + offa;
            const int nrow = min(RP, nrows - c * RP);
            if (nrow == RP && c > 0) {
#pragma unroll
                for (int r = 0; r < RP; ++r) {
                    const double A = st[r * 32], cc = stc[r * 32], q = st[2 * SV + r * 32], a = sta[r * 32];
                    const double R = st[4 * SV + r * 32];
                    double va, vb, vz;
                    elim2_row(S, e, cc, q, a, A, R, va, vb, vz);
                    e = A;
                    st3_if(outl, al + o, va, be + o, vb, zz + o, vz);
                    o += step;
                }
            } else {
                for (int r = 0; r < nrow; ++r) {
                    const double A = st[r * 32], cc = stc[r * 32], q = st[2 * SV + r * 32], a = sta[r * 32];
                    const double R = st[4 * SV + r * 32];
                    double va, vb, vz;
                    elim2_row(S, e, cc, q, a, A, R, va, vb, vz);
                    e = A;
                    st3_if(outl && (c * RP + r) > 0, al + o, va, be + o, vb, zz + o, vz);
                    o += step;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + s);
        }
        double va, vb, vz;
        elim2_flush(S, va, vb, vz);
        st3_if(outl, al + o, va, be + o, vb, zz + o, vz);
    }
}

// ---------------------------------------------------------------------------------------------
// x forward, two-sided, warp-specialised.  One CTA per SM with 4 sub-problems q = warp & 3: two adjacent
// blocks of XW_R rows x two halves (half 0: columns 0 .. mid-1 ascending, half 1: columns nx-1 .. mid
// descending; see yfwd_ws_kernel for the two-sided scheme).  Per sub-problem: one consumer warp (lane <->
// row of the block, marches along the lines) and NP producer warps.  Producers work with lanes ALONG the
// lines (lane <-> column, coalesced loads, x-neighbours by shuffle; only x-neighbours are needed,
// PAPER.md:748) on tiles of 28 columns, split rows r = pw, pw+NP, ... between them, and write, transposed,
// into two ring slots of XW_CK = 14 columns each ([plane][column][XW_LD]: conflict-free for the producers'
// half-warps and for the consumer).  Coefficients go out transposed ([i][j]) so the consumer's stores are coalesced.
//
// What the ring carries: per column the scaled partials (A, p1, p2) of the FORWARD face in marching order (the face
// towards the next column the consumer will eliminate) and the right-hand side w -- 4 planes.  The consumer keeps the
// previous column's face in registers and forms the bands c = -(A + p1'), q = (1 + p1) - p2', a = p2 - A' itself
// (primes: backward face).  Storing faces instead of finished bands (5 planes) saves the producers six shuffles and
// four additions per row and a fifth of the ring (x forward 0.58 -> 0.52 ms at 8192^2).  Ring depth: three slots
// (1.5 tiles).  Four slots (two whole tiles, which the smaller planes would allow) remove the waiting of producers and
// consumer for each other but were measured SLOWER (0.67 ms): the producers' row loads are unaligned 256-byte
// segments that overlap between neighbouring tiles and live on the L1 cache, and 208 KB of shared memory leave too
// little of it (two slots, 104 KB: 0.53 ms).  The next tile's rows are therefore prefetched into L1 while the current
// one is assembled (TF_XW_PREFETCH: 0.52 -> 0.50 ms; the first use of a tile's loads had 12 % of all stall samples).
// For half 1 (descending columns) lane i-1 writes its face i-1/2 into column i's position with p1, p2 swapped and
// negated, which is the same formula in the reversed system.
// ---------------------------------------------------------------------------------------------
#ifndef XW_RECOMPUTE_C1
#define XW_RECOMPUTE_C1 1
#endif
#ifndef TF_XW_PREFETCH
#define TF_XW_PREFETCH 1
#endif
#ifndef TF_ROTATE_X
#define TF_ROTATE_X 1
#endif
constexpr int XW_CT = 28;            // columns per producer tile (32 lanes minus 2 halo lanes each side)
constexpr int XW_CK = 14;            // columns per ring slot
constexpr int XW_R = 28;             // rows per block
constexpr int XW_LD = 29;            // slot row pitch in doubles (odd)

template <int N, int M, int NP, int NCH, int NSUB>
__global__ void __launch_bounds__(32 * fwd_warps(NSUB, NP), 1)
xfwd_ws_kernel(Params P, Dir DX, int mid, const double* __restrict__ u, const double* __restrict__ w,
               double* __restrict__ alT, double* __restrict__ beT, double* __restrict__ zzT, Gate gate)
{
    if (gate_closed(gate)) return;
    if (gate.s) DX = dir_of(__ldcg(gate.s), P.dx);
    constexpr int SV = XW_CK * XW_LD;                 // doubles per value plane of a slot
    constexpr int NPL = 4;                            // planes per slot: A, p1, p2 of the forward face, right-hand side
    constexpr size_t RING = (size_t)NCH * NPL * SV * 8 + 16 * NCH;
    constexpr int NRMAX = (XW_R + NP - 1) / NP;       // rows per producer
    extern __shared__ __align__(16) unsigned char raw[];
    const unsigned FULL = 0xffffffffu;
    const int nx = P.nx, ny = P.ny;
    const int warp = uniform_warp_idx(), lane = threadIdx.x & 31;
    int role, q;                                      // 0: consumer, 1..NP: producers; team q (see yfwd_ws_kernel)
    bool idle = false;
    if (fwd_sp0(NSUB)) {
        if (warp % 4 == 0) { role = 0; q = warp / 4; idle = warp / 4 >= NSUB; }
        else { const int p = warp - warp / 4 - 1; q = p % NSUB; role = 1 + p / NSUB; idle = role > NP; }
        if (idle) { role = 1; q = 0; }
    } else {
        role = warp / NSUB;
        q = TF_ROTATE_X ? (warp % NSUB + NSUB * NP - role) % NSUB : warp % NSUB;
    }
    double* sm = reinterpret_cast<double*>(raw + q * RING);          // [NCH][NPL][CK][LD]
    uint64_t* full = reinterpret_cast<uint64_t*>(raw + q * RING + (size_t)NCH * NPL * SV * 8);
    uint64_t* empty = full + NCH;
    if (role == 0 && lane == 0) {
#pragma unroll
        for (int s = 0; s < NCH; ++s) { mbar_init(full + s, NP); mbar_init(empty + s, 1); }
        mbar_fence_init();
    }
    __syncthreads();
    if (idle) return;
    constexpr int SPC = NSUB >= 2 ? NSUB / 2 : 1;     // row blocks per CTA; NSUB = 1: blockIdx.x = 2 block + half
    const int j0 = (NSUB >= 2 ? SPC * (int)blockIdx.x + (q % SPC) : (int)blockIdx.x / 2) * XW_R;
    if (j0 >= ny) return;
    const int dir = NSUB >= 2 ? q / SPC : (int)blockIdx.x % 2;
    const int ncols = dir ? nx - mid : mid;           // columns of this half
    const int ntile = (ncols + XW_CT - 1) / XW_CT;
    const int imin = dir ? mid : 0, imax = dir ? nx : mid;

    if (role > 0) {
        // ------------------------------------------------------------------ producer pw: rows pw, pw+NP, ... of the block
        const int pw = role - 1;
        size_t rowoff[NRMAX];
#pragma unroll
        for (int k = 0; k < NRMAX; ++k) rowoff[k] = (size_t)min(j0 + pw + k * NP, ny - 1) * nx;
        // The lane of column i computes face i+1/2.  Half 0 stores it at its own column (marching position lane-2);
        // half 1 stores it, as the forward face of column i+1, at marching position 29-(lane+1) = 28-lane.
        const int kk = dir ? XW_CT - lane : lane - 2;
        const bool lane_ok = (kk >= 0) && (kk < XW_CT);      // lanes 2..29 (half 0), 1..28 (half 1)
        const int slot_sel = lane_ok ? kk / XW_CK : 0;       // first or second slot of the tile
        const int kc = lane_ok ? kk % XW_CK : 0;             // column within the slot
        for (int t = 0; t < ntile; ++t) {
            const int ilo = dir ? nx - (t + 1) * XW_CT : t * XW_CT;       // the tile is columns ilo .. ilo+27
            const int i = ilo - 2 + lane;
            const int ic = ghost(i, nx);
            const bool face_ok = (i >= 0) && (i <= nx - 2);
            const int idst = i + dir;                         // the column whose ring position this lane fills
            const bool col_ok = lane_ok && (idst >= imin) && (idst < imax);
            double hq[NRMAX], wq[NRMAX];
#pragma unroll
            for (int k = 0; k < NRMAX; ++k) {
                hq[k] = u[rowoff[k] + ic];
                wq[k] = col_ok ? w[rowoff[k] + idst] : 0.0;
            }
#if TF_XW_PREFETCH
            if (t + 1 < ntile) {                              // pull the next tile's rows into L1 while this one is assembled
                const int in = (dir ? ilo - XW_CT : ilo + XW_CT) - 2 + lane;
                const int icn = ghost(in, nx), iwn = clampi(in + dir, 0, nx - 1);
#pragma unroll
                for (int k = 0; k < NRMAX; ++k) {
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(u + rowoff[k] + icn));
                    asm volatile("prefetch.global.L1 [%0];" ::"l"(w + rowoff[k] + iwn));
                }
            }
#endif
            const int g0 = 2 * t, g1 = 2 * t + 1;             // global slot numbers of this tile
            mbar_wait(empty + g0 % NCH, ((g0 / NCH) & 1) ^ 1);
            mbar_wait(empty + g1 % NCH, ((g1 / NCH) & 1) ^ 1);
            double* st = sm + (size_t)((slot_sel ? g1 : g0) % NCH) * NPL * SV + kc * XW_LD;
            // one row of the tile; INTERIOR: every face of the tile is an interior, unfolded face and every
            // column belongs to this half -- no boundary selects (all tiles but the first, last and the split one)
            auto row = [&](auto interior_tag, int k) {
                constexpr bool INTERIOR = decltype(interior_tag)::value;
                const int r = pw + k * NP;
                const double h0 = hq[k];
                const double hm1 = __shfl_up_sync(FULL, h0, 1);
                const double hp1 = __shfl_down_sync(FULL, h0, 1), hp2 = __shfl_down_sync(FULL, h0, 2);
                const Cell c0 = cell_functions<N, M>(h0, P);
                Cell c1;
                if (XW_RECOMPUTE_C1 && N >= 0) {
                    // power-law Pi: recomputing the neighbour's cell (10 fp64) is cheaper than 8 shuffles -- the LSU
                    // pipe, not fp64, bounds this kernel; the NLC / polymer cells (tanh, high powers) are shuffled
                    c1 = cell_functions<N, M>(hp1, P);
                } else {
                    c1.f0 = __shfl_down_sync(FULL, c0.f0, 1); c1.f1 = __shfl_down_sync(FULL, c0.f1, 1);
                    c1.g0 = __shfl_down_sync(FULL, c0.g0, 1); c1.g1 = __shfl_down_sync(FULL, c0.g1, 1);
                }
                Face fp = face_partials(hm1, hp2, hp1 - h0, c0.f0 + c1.f0, c0.f1 + c1.f1, c0, c1, DX);
                if (!INTERIOR) {
                    if (i == 0) fp.p1 -= fp.A;
                    if (i == nx - 2) fp.p2 += fp.A;
                    if (!face_ok) { fp.A = 0.0; fp.p1 = 0.0; fp.p2 = 0.0; }
                }
                if (INTERIOR ? lane_ok : col_ok) {
                    st[r] = fp.A;
                    st[SV + r] = dir ? -fp.p2 : fp.p1;
                    st[2 * SV + r] = dir ? -fp.p1 : fp.p2;
                    st[3 * SV + r] = wq[k];
                }
            };
            const bool interior = (ilo >= 3) && (ilo + XW_CT + 2 <= nx - 2) && (ilo >= imin) && (ilo + XW_CT <= imax);
            if (interior) {
#pragma unroll
                for (int k = 0; k < NRMAX; ++k)
                    if (pw + k * NP < XW_R) row(std::true_type{}, k);
            } else {
#pragma unroll
                for (int k = 0; k < NRMAX; ++k)
                    if (pw + k * NP < XW_R) row(std::false_type{}, k);
            }
            __syncwarp();
            if (lane == 0) { mbar_arrive(full + g0 % NCH); mbar_arrive(full + g1 % NCH); }
        }
    } else {
        // ------------------------------------------------------------------ consumer: lane <-> row j0 + lane
        const int j = j0 + lane;
        const int rowok = (lane < XW_R && j < ny) ? 1 : 0;
        Elim2 S = elim2_init();
        double Ba = 0.0, B1 = 0.0, B2 = 0.0;              // backward face: the boundary face before the first column carries nothing
        const int step = dir ? -ny : ny;
        int o = (dir ? nx : -1) * ny + j;                 // the column before the first one
        const int lr = min(lane, XW_R - 1);               // lanes beyond the block read a valid row (results unused)
        for (int g = 0; g < 2 * ntile; ++g) {
            const int s = g % NCH;
            mbar_wait(full + s, (g / NCH) & 1);
            const double* st = sm + (size_t)s * NPL * SV + lr;
            const int ncol = min(XW_CK, ncols - g * XW_CK);
            // one column: bands from the forward face (ring) and the backward face (registers), then the recurrence
            auto column = [&](int c, int pred) {
                const double Fa = st[c * XW_LD], F1 = st[SV + c * XW_LD], F2 = st[2 * SV + c * XW_LD];
                const double R = st[3 * SV + c * XW_LD];
                const double cc = -(Fa + B1), qq = (1.0 + F1) - B2, a = F2 - Ba;
                double va, vb, vz;
                elim2_row(S, Ba, cc, qq, a, Fa, R, va, vb, vz);
                Ba = Fa; B1 = F1; B2 = F2;
                st3_if(pred, alT + o, va, beT + o, vb, zzT + o, vz);
                o += step;
            };
            if (ncol == XW_CK && g > 0) {
#pragma unroll
                for (int c = 0; c < XW_CK; ++c) column(c, rowok);
            } else {
                for (int c = 0; c < ncol; ++c) column(c, rowok && (g * XW_CK + c) > 0);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + s);
        }
        double va, vb, vz;
        elim2_flush(S, va, vb, vz);
        st3_if(rowok, alT + o, va, beT + o, vb, zzT + o, vz);
    }
}

}  // namespace tf
