// bt_wyz.cuh -- compact-WY back-transformation on the FP64 tensor cores, COMPLEX FP64 (sm_100a).
// Same algorithm and fragment chaining as bt_wy.cuh; every complex product is four real DMMAs.
//
//      H_7 .. H_0 = I - V T V^H,  T lower triangular, T[j][j] = tau_j,
//      T[j][:j] = -tau_j (v_j^H V[:, :j]) T[:j, :j]                    (R2: tau as stored, v^H in the dot)
//      D^T = x^T conj(V):  Dr = xr Vr + xi Vi,  Di = xi Vr - xr Vi      (four accumulators, 4 chains)
//      Y = V (-T)  (prepass, W x 8 complex):  the update operand, so no separate T product
//      x^T += D^T Y^T:     xr += Dr Yr - Di Yi,  xi += Dr Yi + Di Yr
// Registers hold x planar (real and imaginary fragments apart); global memory and shared memory
// stay interleaved (re, im): one LDS.128 / LDG.128 = one complex element.  Interleaved 16-byte
// elements keep the skewed rows of VA 16-byte aligned, so VA is staged with one bulk copy (TMA
// engine) per reflector and YB with one more.
#pragma once
#include "bt_wy.cuh"

namespace elpa2bt {

template <int NBW_>
struct WyzCfg {
    static constexpr int NBW = NBW_;
    static constexpr int NB8 = NBW / 8;               // 8-row blocks per chase block
    static constexpr int NT = NBW / 8 + 1;            // 8-row tiles in the window
    static constexpr int W = 8 * NT;                  // window rows
    static constexpr int NW = 8;                      // warps per CTA
    static constexpr int NGMAX = (NBW <= 64) ? 2 : 1; // most 8-column slabs per warp
    static constexpr int NS = (NBW <= 64) ? 8 : 4;    // ring stages
    static constexpr int LGNS = (NBW <= 64) ? 3 : 2;
    static constexpr int LAG = NS / 2;                // staging waits for the block LAG iterations back
    // element = 2 doubles.  Row strides padded by one element: rows gq and gq+1 of a quarter-warp
    // then differ by 4 banks (W*4 and 8*4 words are multiples of 32)
    static constexpr int SA = W + 1;                  // VA[i][w] row stride (elements)
    static constexpr int SB = 9;                      // VB[w][i] row stride (elements)
    static constexpr int VA_OFF = 0;                  // offsets in doubles; VA[i][w] = V
    static constexpr int YB_OFF = 2 * 8 * SA;         // YB[w][j] = (V (-T))[w][j]
    static constexpr int YBLK = 2 * W * SB;           // doubles of scratch per block (its YB image, padded rows)
    static constexpr int STAGE_DOUBLES = ((YB_OFF + YBLK + 15) / 16) * 16;
    static constexpr int PW = (NBW <= 64) ? 4 : 2;    // warps (= blocks) per CTA of the prepass kernel
    static constexpr int OFF_BAR = NS * STAGE_DOUBLES * 8;
    static constexpr int SMEM_BYTES = OFF_BAR + 2 * NS * 8;
    static_assert((YB_OFF * 8) % 16 == 0 && (YBLK * 8) % 16 == 0, "16-byte aligned sections");
    static_assert(SMEM_BYTES <= 227 * 1024, "shared memory");
};

// ---- prepass: Y = V (-T) of every block, as the padded YB[w][j] image (interleaved complex) --------------
template <int NBW>
__global__ void __launch_bounds__(WyzCfg<NBW>::PW * 32) wyz_prepass_kernel(int64_t N, const double *__restrict__ hh_v,
                                                                           const double *__restrict__ hh_tau,
                                                                           double *__restrict__ yb, int64_t kb)
{
    using C = WyzCfg<NBW>;
    constexpr int W = C::W, SV = W + 1;               // Vs row stride (elements)
    __shared__ double Sm[C::PW][128];
    __shared__ double Vs[C::PW][8 * SV * 2];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int gq = lane >> 2, r = lane & 3;
    const int64_t k = kb + blockIdx.y;
    const int64_t bhi = wy_bhi(N);
    const int64_t nblk = bhi - (k * C::NB8) + 1;
    const int64_t j = (int64_t)blockIdx.x * C::PW + warp;
    if (j >= nblk) return;
    const int64_t b = bhi - j;
    const int64_t FN1 = hh_F(N - 1, C::NBW);
    const int64_t slot = wy_slot<C::NBW>(N, FN1, k, b, gq);
    double taur = 0.0, taui = 0.0;
    if (slot >= 0) {
        taur = hh_tau[2 * slot];
        taui = hh_tau[2 * slot + 1];
    }
    // S = V^H V:  Sr = Vr^T Vr + Vi^T Vi,  Si = Vr^T Vi - Vi^T Vr
    double a0 = 0.0, a1 = 0.0, b0 = 0.0, b1 = 0.0, p0 = 0.0, p1 = 0.0, q0 = 0.0, q1 = 0.0;
#pragma unroll
    for (int c = 0; c < W / 4; ++c) {
        const int rl = 4 * c + r - (7 - gq);
        double vr = 0.0, vi = 0.0;
        if (slot >= 0 && rl >= 0 && rl < NBW) {
            const double2 v2 = *reinterpret_cast<const double2 *>(hh_v + (slot * NBW + rl) * 2);
            vr = v2.x;
            vi = v2.y;
        }
        *reinterpret_cast<double2 *>(&Vs[warp][(gq * SV + 4 * c + r) * 2]) = make_double2(vr, vi);
        dmma884(a0, a1, vr, vr, a0, a1);
        dmma884(b0, b1, vi, vi, b0, b1);
        dmma884(p0, p1, vr, vi, p0, p1);
        dmma884(q0, q1, vi, vr, q0, q1);
    }
    // S[m = gq][n = 2r + {0,1}]
    Sm[warp][(gq * 8 + 2 * r) * 2] = a0 + b0;
    Sm[warp][(gq * 8 + 2 * r) * 2 + 1] = p0 - q0;
    Sm[warp][(gq * 8 + 2 * r + 1) * 2] = a1 + b1;
    Sm[warp][(gq * 8 + 2 * r + 1) * 2 + 1] = p1 - q1;
    __syncwarp();
    const int l = lane & 7;
    double tr[8], ti[8];
#pragma unroll
    for (int jj = 0; jj < 8; ++jj) {
        const double tjr = __shfl_sync(0xffffffffu, taur, 4 * jj);
        const double tji = __shfl_sync(0xffffffffu, taui, 4 * jj);
        double ar = 0.0, ai = 0.0;
#pragma unroll
        for (int i = 0; i < jj; ++i) {
            const double sr = Sm[warp][(jj * 8 + i) * 2], si = Sm[warp][(jj * 8 + i) * 2 + 1];
            ar = fma(sr, tr[i], ar);
            ar = fma(-si, ti[i], ar);
            ai = fma(sr, ti[i], ai);
            ai = fma(si, tr[i], ai);
        }
        // -tau_j * acc
        const double mr = -(tjr * ar - tji * ai), mi = -(tjr * ai + tji * ar);
        tr[jj] = (jj == l) ? tjr : (jj > l ? mr : 0.0);
        ti[jj] = (jj == l) ? tji : (jj > l ? mi : 0.0);
    }
    __syncwarp();
    if (lane < 8) {
#pragma unroll
        for (int jj = 0; jj < 8; ++jj) {                                   // Sm = -T, row-major [i][j]
            Sm[warp][(jj * 8 + l) * 2] = -tr[jj];
            Sm[warp][(jj * 8 + l) * 2 + 1] = -ti[jj];
        }
    }
    __syncwarp();
    // Y[w][j] = sum_i V[w][i] T'[i][j], T' = -T:  Yr = Vr Tr' - Vi Ti',  Yi = Vr Ti' + Vi Tr'
    double tbr[2], tbi[2];
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        tbr[c] = Sm[warp][((r + 4 * c) * 8 + gq) * 2];
        tbi[c] = Sm[warp][((r + 4 * c) * 8 + gq) * 2 + 1];
    }
    double *out = yb + (wy_base(N, C::NBW, k) + j) * C::YBLK;
#pragma unroll
    for (int tt = 0; tt < C::NT; ++tt) {
        double yr0 = 0.0, yr1 = 0.0, yi0 = 0.0, yi1 = 0.0;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const double2 v2 = *reinterpret_cast<const double2 *>(&Vs[warp][((r + 4 * c) * SV + 8 * tt + gq) * 2]);
            dmma884(yr0, yr1, v2.x, tbr[c], yr0, yr1);
            dmma884(yr0, yr1, -v2.y, tbi[c], yr0, yr1);
            dmma884(yi0, yi1, v2.x, tbi[c], yi0, yi1);
            dmma884(yi0, yi1, v2.y, tbr[c], yi0, yi1);
        }
        double *o = out + ((8 * tt + gq) * C::SB + 2 * r) * 2;
        *reinterpret_cast<double2 *>(o) = make_double2(yr0, yi0);
        *reinterpret_cast<double2 *>(o + 2) = make_double2(yr1, yi1);
    }
    // the padding column (j = 8) of the image is never read; it is zeroed once so that the bulk copy moves
    // defined bytes
    for (int w = lane; w < W; w += 32) *reinterpret_cast<double2 *>(out + (w * C::SB + 8) * 2) = make_double2(0.0, 0.0);
}

// ---- staging one block (whole warp) ---------------------------------------------------------------------
// bulk copies (TMA engine) only: one per reflector for VA[i][7 - i + ..] (interleaved 16-byte elements keep
// the skewed rows 16-byte aligned) and one for the YB image the prepass wrote.  Full barrier: one arrival
// (lane 0) carrying the byte count.
template <class C>
__device__ __forceinline__ void wyz_stage(const WyArgs &a, double *stage, uint32_t bar_full, int64_t k, int64_t b,
                                          int64_t id, int64_t FN1, int lane)
{
    constexpr int NBW = C::NBW;
    const int i8 = lane & 7;
    const int64_t slot = wy_slot<C::NBW>(a.N, FN1, k, b, i8);
    const unsigned valid = __ballot_sync(0xffffffffu, slot >= 0) & 0xffu;
    if (lane == 0) {
        mbar_arrive_expect_tx(bar_full, (uint32_t)__popc(valid) * NBW * 16u + C::YBLK * 8u);
        bulk_g2s(smem_u32(stage + C::YB_OFF), a.tn + id * C::YBLK, C::YBLK * 8u, bar_full);
    }
    __syncwarp();
    if (lane < 8 && slot >= 0)
        bulk_g2s(smem_u32(stage + C::VA_OFF + (i8 * C::SA + 7 - i8) * 2), a.hh_v + slot * NBW * 2, NBW * 16u, bar_full);
}

// ---- tile I/O: rows row0 + 2r + {0,1} of this lane's column (interleaved in memory, planar in regs) ----
template <bool CG = false>
__device__ __forceinline__ void wyz_load2(const WyArgs &a, const int64_t nrow, const double *colp, bool colok, int64_t row, double &xr0,
                                          double &xr1, double &xi0, double &xi1)
{
    xr0 = xr1 = xi0 = xi1 = 0.0;
    if (!colok || row >= nrow) return;
    const double2 v = CG ? __ldcg(reinterpret_cast<const double2 *>(colp + 2 * row))
                         : *reinterpret_cast<const double2 *>(colp + 2 * row);
    xr0 = v.x;
    xi0 = v.y;
    if (row + 1 < nrow) {
        const double2 w = CG ? __ldcg(reinterpret_cast<const double2 *>(colp + 2 * row + 2))
                             : *reinterpret_cast<const double2 *>(colp + 2 * row + 2);
        xr1 = w.x;
        xi1 = w.y;
    }
}
__device__ __forceinline__ void wyz_store2(const WyArgs &a, const int64_t nrow, double *colp, bool colok, int64_t row, double xr0,
                                           double xr1, double xi0, double xi1)
{
    if (!colok || row >= nrow) return;
    *reinterpret_cast<double2 *>(colp + 2 * row) = make_double2(xr0, xi0);
    if (row + 1 < nrow) *reinterpret_cast<double2 *>(colp + 2 * row + 2) = make_double2(xr1, xi1);
}

// ---- a warp with NG slabs of 8 columns -------------------------------------------------------------------
// Same structure as wy_consume (bt_wy.cuh): CP = chain-parallel mode (a.P warps per slab, NG = 1).
template <class C, int NG, bool CP, bool RG>
__device__ __forceinline__ void wyz_consume(const WyArgs &a, unsigned char *smem, const int lane, const int grp,
                                            const int member, const int nmem, const int64_t col0, const int64_t slab)
{
    constexpr int NT = C::NT, NBW = C::NBW;
    const int P = CP ? a.P : 1;
    const int lgs = CP ? C::LGNS - 1 : C::LGNS;        // P = 2 is the only chain-parallel width here
    const int NSP = 1 << lgs, LAG = NSP >> 1;
    double *ring = reinterpret_cast<double *>(smem) + (size_t)grp * NSP * C::STAGE_DOUBLES;
    const uint32_t bar_full = smem_u32(smem + C::OFF_BAR) + 8 * grp * NSP;
    const uint32_t bar_empty = bar_full + C::NS * 8;
    const int gq = lane >> 2, r = lane & 3;
    const int64_t N = a.N;
    const int64_t K0 = wy_nchains(N, C::NBW);
    const int64_t bhi = wy_bhi(N);                      // numbering of the blocks (scratch ids) is global
    // RG = false (the whole matrix) keeps every bound a compile-time function of N: the code of the full launch
    const int64_t btop = RG ? a.b_top : bhi;
    const int64_t nrow = RG ? a.row_end : N;            // rows >= nrow are not in memory
    const int64_t kb = RG ? a.kb : 0, ke = RG ? a.ke : K0;                       // first block of every chain in this launch (bt_wy.cuh)
    const int64_t FN1 = hh_F(N - 1, C::NBW);

    // this lane's columns: col0 + 8g + gq, g = 0 .. NG-1 (ldq counts complex elements)
    double *const cb = a.q + (col0 + gq < a.nev ? col0 + gq : 0) * a.ldq * 2;
    const int64_t ldq8 = a.ldq << 4;
    const int64_t ncolrem = a.nev - col0 - gq;          // column g is valid iff 8g < ncolrem
    const bool fastio = col0 + 8 * NG <= a.nev;         // warp-uniform: every column of the warp exists

    auto bbot = [&](int64_t k) { return (RG && k * C::NB8 < a.b_bot) ? a.b_bot : k * C::NB8; };   // last block of chain k here
    int64_t pk = kb + grp, pb = btop;                 // staging cursor: block it + NSP - LAG of this ring
    auto advance = [&]() {
        if (pb > bbot(pk)) {
            --pb;
        } else {
            pk += P;
            pb = btop;
        }
    };
    auto stage_cursor = [&](uint32_t st) {
        wyz_stage<C>(a, ring + st * C::STAGE_DOUBLES, bar_full + 8 * st, pk, pb, wy_base(N, C::NBW, pk) + (bhi - pb), FN1,
                     lane);
    };
    for (int i = 0; i < NSP - LAG; ++i) {
        if (member == 0 && pk < ke) stage_cursor((uint32_t)i);
        advance();
    }

    // tile 0 alternates between TA and TB (refilled two blocks ahead, bt_wy.cuh); [..][0..1] = real
    // parts of rows 2r, 2r+1, [..][2..3] = imaginary parts
    double Xr[NG][NT + 1][2], Xi[NG][NT + 1][2], TA[NG][4], TB[NG][4];
    uint32_t it = 0;
    int duty = 0;
    for (int64_t k = kb + grp; k < ke; k += P) {
        const int64_t blo = bbot(k);
        const uint32_t *prev = (CP && k > kb) ? a.prog + slab * K0 + (k - 1) : nullptr;
        uint32_t *mine = CP ? a.prog + slab * K0 + k : nullptr;
        uint32_t known = 0;
        auto wait_prev = [&](int64_t b) {
            if (CP && prev) {
                const uint32_t need = (uint32_t)(btop - b + NBW / 8 + 1);
                while (known < need) known = prog_read(prev);
            }
        };
        auto load_tile0 = [&](int64_t b, double (&T0)[NG][4]) {
            if (b < blo) return;
            wait_prev(b);
#pragma unroll
            for (int g = 0; g < NG; ++g)
                wyz_load2<CP>(a, nrow, cb + g * ldq8, 8 * g < ncolrem, (b << 3) + 2 * r, T0[g][0], T0[g][1], T0[g][2], T0[g][3]);
        };
        auto do_block = [&](const int64_t b, double (&T0)[NG][4]) {
            if (duty == member) {
                if (pk < ke) {
                    const uint32_t st = (it + NSP - LAG) & (NSP - 1);
                    if (it >= (uint32_t)LAG) mbar_wait(bar_empty + 8 * st, ((it - LAG) >> lgs) & 1);
                    stage_cursor(st);
                }
            }
            advance();
            duty = (duty + 1 == nmem) ? 0 : duty + 1;

            const uint32_t st = it & (NSP - 1), ph = (it >> lgs) & 1;
            mbar_wait(bar_full + 8 * st, ph);
            const double *stage = ring + st * C::STAGE_DOUBLES;
            const double *va = stage + C::VA_OFF + (gq * C::SA + 2 * r) * 2;   // + (8t + e) * 2
            const double *vb = stage + C::YB_OFF + (gq * C::SB + 2 * r) * 2;   // + 8t * SB * 2 + e * 2

            // --- D^T = x^T conj(V) with three real products instead of four (the 3M form of a complex product):
            //     P1 = xr Vr, P2 = xi Vi, P3 = (xr + xi)(Vr - Vi)  =>  Dr = P1 + P2, Di = P3 - P1 + P2.
            //     The two operand sums are one DADD each per k-chunk (same FP64 pipe: 2 cycles against the 16 of
            //     the DMMA they replace); normwise the rounding error is that of the four-product form.
            //     Two accumulator sets (e = 0 / 1): six independent DMMA chains per slab.
            double P1[NG][2][2], P2[NG][2][2], P3[NG][2][2];
#pragma unroll
            for (int g = 0; g < NG; ++g)
#pragma unroll
                for (int e = 0; e < 2; ++e)
                    P1[g][e][0] = P1[g][e][1] = P2[g][e][0] = P2[g][e][1] = P3[g][e][0] = P3[g][e][1] = 0.0;
#pragma unroll
            for (int tt = 0; tt < NT; ++tt) {
                const int t = (tt + 1) % NT;
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const double2 v2 = *reinterpret_cast<const double2 *>(va + (8 * t + e) * 2);
                    const double vd = v2.x - v2.y;
#pragma unroll
                    for (int g = 0; g < NG; ++g) {
                        const double xr = t ? Xr[g][t][e] : T0[g][e], xi = t ? Xi[g][t][e] : T0[g][2 + e];
                        dmma884(P1[g][e][0], P1[g][e][1], xr, v2.x, P1[g][e][0], P1[g][e][1]);
                        dmma884(P2[g][e][0], P2[g][e][1], xi, v2.y, P2[g][e][0], P2[g][e][1]);
                        dmma884(P3[g][e][0], P3[g][e][1], xr + xi, vd, P3[g][e][0], P3[g][e][1]);
                    }
                }
            }
            // --- E^T = D^T (T is folded into YB = V (-T)): Er = P1 + P2, Ei = P3 - P1 + P2
            double Er[NG][2], Ei[NG][2], nEi[NG][2];
#pragma unroll
            for (int g = 0; g < NG; ++g)
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    const double p1 = P1[g][0][c] + P1[g][1][c], p2 = P2[g][0][c] + P2[g][1][c], p3 = P3[g][0][c] + P3[g][1][c];
                    Er[g][c] = p1 + p2;
                    Ei[g][c] = (p3 - p1) + p2;
                    nEi[g][c] = -Ei[g][c];
                }
            // --- x^T += E^T Y^T: xr += Er Yr - Ei Yi, xi += Er Yi + Ei Yr; tile t -> registers of t+1
#pragma unroll
            for (int t = NT - 1; t >= 0; --t) {
                const double2 v0 = *reinterpret_cast<const double2 *>(vb + 8 * t * C::SB * 2);
                const double2 v1 = *reinterpret_cast<const double2 *>(vb + 8 * t * C::SB * 2 + 2);
#pragma unroll
                for (int g = 0; g < NG; ++g) {
                    double m0, m1, n0, n1;
                    dmma884(m0, m1, Er[g][0], v0.x, t ? Xr[g][t][0] : T0[g][0], t ? Xr[g][t][1] : T0[g][1]);
                    dmma884(n0, n1, Er[g][0], v0.y, t ? Xi[g][t][0] : T0[g][2], t ? Xi[g][t][1] : T0[g][3]);
                    dmma884(m0, m1, nEi[g][0], v0.y, m0, m1);
                    dmma884(n0, n1, Ei[g][0], v0.x, n0, n1);
                    dmma884(m0, m1, Er[g][1], v1.x, m0, m1);
                    dmma884(n0, n1, Er[g][1], v1.y, n0, n1);
                    dmma884(Xr[g][t + 1][0], Xr[g][t + 1][1], nEi[g][1], v1.y, m0, m1);
                    dmma884(Xi[g][t + 1][0], Xi[g][t + 1][1], Ei[g][1], v1.x, n0, n1);
                }
            }
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(bar_empty + 8 * st);
                if (CP && b < btop) prog_publish(mine, (uint32_t)(btop - b));
            }
            if (fastio && (b << 3) + NBW + 8 <= nrow) {
                // the block lies inside the matrix: no per-access guards (bt_wy.cuh)
                double *pr = cb + 2 * ((b << 3) + 2 * r);
#pragma unroll
                for (int g = 0; g < NG; ++g) {
                    *reinterpret_cast<double2 *>(pr + g * ldq8 + 2 * NBW) = make_double2(Xr[g][NT][0], Xi[g][NT][0]);
                    *reinterpret_cast<double2 *>(pr + g * ldq8 + 2 * NBW + 2) = make_double2(Xr[g][NT][1], Xi[g][NT][1]);
                }
                if (b - 2 >= blo) {
                    wait_prev(b - 2);
                    const double *pl = pr - 32;
#pragma unroll
                    for (int g = 0; g < NG; ++g) {
                        const double2 v = CP ? __ldcg(reinterpret_cast<const double2 *>(pl + g * ldq8))
                                             : *reinterpret_cast<const double2 *>(pl + g * ldq8);
                        const double2 w = CP ? __ldcg(reinterpret_cast<const double2 *>(pl + g * ldq8 + 2))
                                             : *reinterpret_cast<const double2 *>(pl + g * ldq8 + 2);
                        T0[g][0] = v.x;
                        T0[g][2] = v.y;
                        T0[g][1] = w.x;
                        T0[g][3] = w.y;
                    }
                }
            } else {
#pragma unroll
                for (int g = 0; g < NG; ++g)
                    wyz_store2(a, nrow, cb + g * ldq8, 8 * g < ncolrem, (b << 3) + NBW + 2 * r, Xr[g][NT][0], Xr[g][NT][1],
                               Xi[g][NT][0], Xi[g][NT][1]);
                load_tile0(b - 2, T0);
            }
            ++it;
        };

        // the window above tile 0 (zero beyond the matrix; a sub-range launch reads the rows handed over)
#pragma unroll
        for (int g = 0; g < NG; ++g) {
#pragma unroll
            for (int t = 1; t < NT; ++t) {
                if (RG)
                    wyz_load2<CP>(a, nrow, cb + g * ldq8, 8 * g < ncolrem, (btop << 3) + 8 * t + 2 * r, Xr[g][t][0], Xr[g][t][1],
                                  Xi[g][t][0], Xi[g][t][1]);
                else
                    Xr[g][t][0] = Xr[g][t][1] = Xi[g][t][0] = Xi[g][t][1] = 0.0;
            }
            Xr[g][NT][0] = Xr[g][NT][1] = Xi[g][NT][0] = Xi[g][NT][1] = 0.0;
#pragma unroll
            for (int i = 0; i < 4; ++i) TA[g][i] = TB[g][i] = 0.0;
        }
        load_tile0(btop, TA);
        load_tile0(btop - 1, TB);
        for (int64_t b = btop; b >= blo; b -= 2) {
            do_block(b, TA);
            if (b - 1 >= blo) do_block(b - 1, TB);
        }
#pragma unroll
        for (int g = 0; g < NG; ++g)
#pragma unroll
            for (int t = 1; t < NT; ++t)
                wyz_store2(a, nrow, cb + g * ldq8, 8 * g < ncolrem, (blo << 3) + 8 * (t - 1) + 2 * r, Xr[g][t][0], Xr[g][t][1],
                           Xi[g][t][0], Xi[g][t][1]);
        if (CP) {
            __syncwarp();
            if (lane == 0) prog_publish(mine, (uint32_t)(btop - blo + 1));
        }
    }
}

// ---- the kernel --------------------------------------------------------------------------------------------
template <int NBW, bool RG = false>
__global__ void __launch_bounds__(256, 1) bt_wyz_kernel(const WyArgs a)
{
    using C = WyzCfg<NBW>;
    constexpr int NS = C::NS, NW = C::NW, NGMAX = C::NGMAX;
    extern __shared__ __align__(128) unsigned char smem[];
    double *ring = reinterpret_cast<double *>(smem);
    const uint32_t bar_full = smem_u32(smem + C::OFF_BAR);
    const uint32_t bar_empty = bar_full + NS * 8;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t nslab = (a.nev + 7) >> 3;
    const int64_t slab0 = nslab * blockIdx.x / gridDim.x;
    const int nmine = (int)(nslab * (blockIdx.x + 1) / gridDim.x - slab0);
    const int nslot = NW / (a.P > 1 ? a.P : 1);
    const int nact = nmine < nslot ? nmine : nslot;    // members of a ring (P = 1: active warps)

    for (int i = threadIdx.x; i < C::OFF_BAR / 8; i += blockDim.x) ring[i] = 0.0;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (threadIdx.x == 0) {
        for (int i = 0; i < NS; ++i) {
            mbar_init(bar_full + 8 * i, 1);            // lane 0 of the staging warp, with the byte count
            mbar_init(bar_empty + 8 * i, (uint32_t)nact);
        }
        mbar_fence_init();
    }
    __syncthreads();

    if (!RG && a.P > 1) {
        // chain-parallel: NW / P groups of P warps; a group takes nmine / (NW / P) slabs (+1 for the first ones)
        const int grp = warp % a.P, member = warp / a.P, nm = NW / a.P;
        const int base = nmine / nm, extra = nmine % nm;
        const int ng = base + (member < extra ? 1 : 0);
        const int64_t wslab0 = slab0 + (int64_t)member * base + (member < extra ? member : extra);
        if (ng == 0) return;
        if (NGMAX >= 2 && ng == 2)
            wyz_consume<C, (NGMAX >= 2 ? 2 : 1), true, false>(a, smem, lane, grp, member, nact, wslab0 << 3, wslab0);
        else
            wyz_consume<C, 1, true, false>(a, smem, lane, grp, member, nact, wslab0 << 3, wslab0);
        return;
    }
    const int base = nmine / NW, extra = nmine % NW;
    const int ng = base + (warp < extra ? 1 : 0);
    const int64_t wslab0 = slab0 + (int64_t)warp * base + (warp < extra ? warp : extra);
    if (ng == 0) return;
    const int64_t col0 = wslab0 << 3;
    if (NGMAX >= 2 && ng == 2)
        wyz_consume<C, (NGMAX >= 2 ? 2 : 1), false, RG>(a, smem, lane, 0, warp, nact, col0, wslab0);
    else
        wyz_consume<C, 1, false, RG>(a, smem, lane, 0, warp, nact, col0, wslab0);
}

template <int NBW>
size_t wyz_tn_bytes(int64_t N)
{
    return (size_t)wy_nblocks(N, NBW) * WyzCfg<NBW>::YBLK * sizeof(double);
}
template <int NBW>
size_t wyz_scratch_bytes(int64_t N, int64_t nev)
{
    const size_t prog = (size_t)((nev + 7) >> 3) * (size_t)wy_nchains(N, NBW) * sizeof(uint32_t);
    return wyz_tn_bytes<NBW>(N) + ((prog + 255) & ~(size_t)255);
}

template <int NBW>
size_t wyz_tn_bytes_range(int64_t N, int64_t kb, int64_t ke)
{
    return (size_t)(wy_base(N, NBW, ke) - wy_base(N, NBW, kb)) * WyzCfg<NBW>::YBLK * sizeof(double);
}

// rg: sub-range launch (bt_wy.cuh WyRange; ldq and the row shift count complex elements)
template <int NBW>
cudaError_t launch_wyz(int64_t N, int64_t nev, const double *hh_v, const double *hh_tau, double *q, int64_t ldq,
                       int nsm, void *scratch, cudaStream_t st, int force_P = 0, const WyRange &rg = WyRange())
{
    using C = WyzCfg<NBW>;
    auto kern = rg.whole() ? bt_wyz_kernel<NBW, false> : bt_wyz_kernel<NBW, true>;
    {
        cudaError_t e = set_max_smem((const void *)kern, C::SMEM_BYTES);
        if (e != cudaSuccess) return e;
    }
    const int64_t K0 = wy_nchains(N, C::NBW);
    const int64_t nslab = (nev + 7) >> 3;
    WyArgs a;
    wy_range_resolve(rg, N, NBW, a.kb, a.ke, a.b_top, a.b_bot, a.row_end);
    if (a.ke <= a.kb) return cudaSuccess;
    if (!rg.whole()) force_P = 1;
    const size_t tn_bytes = rg.whole() ? wyz_tn_bytes<NBW>(N) : wyz_tn_bytes_range<NBW>(N, a.kb, a.ke);
    double *tn_scratch = (double *)scratch - wy_base(N, NBW, a.kb) * C::YBLK;
    uint32_t *prog = (uint32_t *)((char *)scratch + tn_bytes);
    const WyPlan pl = wy_plan(true, NBW, N, nev, nsm, force_P, 8);
    const int P = pl.P;
    cudaError_t e;
    if (P > 1) {
        e = cudaMemsetAsync(prog, 0, (size_t)nslab * K0 * sizeof(uint32_t), st);
        if (e != cudaSuccess) return e;
    }
    const dim3 pgrid((unsigned)((wy_bhi(N) + C::PW) / C::PW), (unsigned)(a.ke - a.kb));
    wyz_prepass_kernel<NBW><<<pgrid, C::PW * 32, 0, st>>>(N, hh_v, hh_tau, tn_scratch, a.kb);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const int64_t grid = pl.grid;
    a.N = N;
    a.nev = nev;
    a.ldq = ldq;
    a.hh_v = hh_v;
    a.hh_tau = hh_tau;
    a.q = q - 2 * rg.row0;
    a.tn = tn_scratch;
    a.prog = prog;
    a.align16 = 1;
    a.P = P;
    kern<<<(unsigned)grid, 256, C::SMEM_BYTES, st>>>(a);
    return cudaGetLastError();
}

}  // namespace elpa2bt
