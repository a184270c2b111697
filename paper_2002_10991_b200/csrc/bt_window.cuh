// bt_window.cuh -- register-resident sliding-window back-transformation kernel (sm_100a).
//
// What it computes: include/elpa2_bt.h (Eq. 6d, Eq. 8).
// How:
//  * Columns of q are independent: a warp owns CW columns for the whole call; CTAs
//    never communicate.
//  * Order: chain-major (k ascending outermost, s descending inside), a dependency-respecting
//    reorder of "reverse generation order" (R5).  Along one chain the
//    nbw-row window moves up by one row per reflector.
//  * The window lives in REGISTERS.  Register slot j holds the row congruent to j (mod nbw), so
//    registers never move: each step exactly one slot retires its row (bottom of the window) and
//    admits the new top row (PAPER.md:174 step 3).  Lane l of the LPC lanes that share a column
//    holds slots 16l..16l+15; the rotation is absorbed by the ADDRESS of v in shared memory
//    (dynamic), not by register indices (static after unrolling 16 steps).
//  * v^H x (PAPER.md:172 step 2a): 16 FMAs per lane and column, then log2(LPC) warp-shuffle
//    stages; x <- x - tau d v (PAPER.md:173 step 2b): 16 FMAs.
//  * Reflectors are staged once per CTA by a producer warp with 1-D bulk copies (TMA engine,
//    UBLKCP) into a ring of 16-reflector blocks guarded by full/empty mbarriers.
//  * Rows enter/leave through per-warp 16-row tiles: cp.async fill of the 16 rows above the
//    window (one full 128-byte line per column), in-place exchange new<->retired during the 16
//    steps, coalesced 16-byte stores of the retired rows.
#pragma once
#include "bt_common.cuh"

namespace elpa2bt {

template <bool CPLX, int NBW_, int CPL_>
struct WinCfg {
    static constexpr int NBW = NBW_;
    static constexpr int LG = (NBW == 32) ? 5 : (NBW == 64) ? 6 : 7;
    static constexpr int CPL = CPL_;                 // columns per lane
    static constexpr int LPC = NBW / 16;             // lanes sharing one column
    static constexpr int NCG = 32 / LPC;             // column groups per warp
    static constexpr int CW = NCG * CPL;             // columns per warp
    static constexpr int EW = CPLX ? 2 : 1;          // doubles per element
    static constexpr int ESZ = 8 * EW;
    static constexpr int TSTRIDE = CPLX ? 17 : 18;   // tile column stride (elements): bank spread
    static constexpr int TILE_BYTES = CW * TSTRIDE * ESZ;
    // v in shared memory: LPC groups of 16 rows, group stride padded by 16 bytes so that the LPC
    // row lanes of a column (which read the same offset of different groups) hit different banks
    static constexpr int GS = 16 + (CPLX ? 1 : 2);    // group stride (elements)
    static constexpr int VS = LPC * GS;               // reflector stride (elements)
    static constexpr int VBLK_BYTES = 16 * VS * ESZ;
    static constexpr int TAU_BYTES = 16 * ESZ;
    static constexpr int NS = (VBLK_BYTES > 16384) ? 3 : 4;   // ring stages
    static constexpr int OFF_TAU = NS * VBLK_BYTES;
    static constexpr int OFF_BAR = OFF_TAU + NS * TAU_BYTES;
    static constexpr int OFF_TILE = OFF_BAR + 2 * NS * 8;
    static_assert(OFF_TILE % 16 == 0, "tile alignment");
    static size_t smem_bytes(int nw) { return (size_t)OFF_TILE + (size_t)nw * 2 * TILE_BYTES; }
};

// ---- tile fill / drain / flush -----------------------------------------------------------------
// Tile buffer: element (c, r) of the warp's CW x 16 block at tile[(c*TSTRIDE + r) * EW].
template <class C, bool CPLX>
__device__ __forceinline__ void tile_fill(const WinArgs &a, double *tile, int64_t col0, int64_t B, int lane)
{
    const int64_t row_base = B << 4;
    if (CPLX || a.align16) {
        constexpr int CE = CPLX ? 1 : 2;          // elements per 16-byte chunk
        constexpr int CPC = 16 / CE;              // chunks per column
#pragma unroll
        for (int t = 0; t < C::CW * CPC / 32; ++t) {
            const int id = lane + 32 * t;
            const int c = id / CPC, ch = id % CPC;
            const int64_t row = row_base + ch * CE, col = col0 + c;
            int64_t nvalid = a.N - row;
            nvalid = nvalid < 0 ? 0 : (nvalid > CE ? CE : nvalid);
            if (col >= a.nev) nvalid = 0;
            const double *src = nvalid ? a.q + (col * a.ldq + row) * C::EW : a.q;
            cp_async16(smem_u32(tile + (c * C::TSTRIDE + ch * CE) * C::EW), src, (uint32_t)nvalid * C::ESZ);
        }
    } else {
#pragma unroll
        for (int t = 0; t < C::CW * 16 / 32; ++t) {
            const int id = lane + 32 * t;
            const int c = id >> 4, r = id & 15;
            const int64_t row = row_base + r, col = col0 + c;
            const bool ok = row < a.N && col < a.nev;
            const double *src = ok ? a.q + col * a.ldq + row : a.q;
            cp_async8(smem_u32(tile + c * C::TSTRIDE + r), src, ok ? 8u : 0u);
        }
    }
}

// store tile rows to global rows [16*Bout, 16*Bout+15] (those < N), columns < nev
template <class C, bool CPLX>
__device__ __forceinline__ void tile_drain(const WinArgs &a, const double *tile, int64_t col0, int64_t Bout, int lane)
{
    const int64_t row_base = Bout << 4;
    if (row_base >= a.N) return;
    if (CPLX || a.align16) {
        constexpr int CE = CPLX ? 1 : 2;
        constexpr int CPC = 16 / CE;
#pragma unroll
        for (int t = 0; t < C::CW * CPC / 32; ++t) {
            const int id = lane + 32 * t;
            const int c = id / CPC, ch = id % CPC;
            const int64_t row = row_base + ch * CE, col = col0 + c;
            if (col < a.nev && row < a.N) {
                const double2 val = *reinterpret_cast<const double2 *>(tile + (c * C::TSTRIDE + ch * CE) * C::EW);
                double *dst = a.q + (col * a.ldq + row) * C::EW;
                if (CPLX || row + 1 < a.N)
                    *reinterpret_cast<double2 *>(dst) = val;
                else
                    *dst = val.x;
            }
        }
    } else {
#pragma unroll
        for (int t = 0; t < C::CW * 16 / 32; ++t) {
            const int id = lane + 32 * t;
            const int c = id >> 4, r = id & 15;
            const int64_t row = row_base + r, col = col0 + c;
            if (col < a.nev && row < a.N) a.q[col * a.ldq + row] = tile[c * C::TSTRIDE + r];
        }
    }
}

// ---- the kernel -------------------------------------------------------------------------------
template <bool CPLX, int NBW, int CPL, int MAXT>
__global__ void __maxnreg__((65536 / MAXT / 8 * 8) > 255 ? 255 : (65536 / MAXT / 8 * 8)) bt_window_kernel(const WinArgs a)
{
    using C = WinCfg<CPLX, NBW, CPL>;
    constexpr int EW = C::EW, LPC = C::LPC, NCG = C::NCG, NS = C::NS;
    extern __shared__ __align__(128) unsigned char smem[];
    double *ring_v = reinterpret_cast<double *>(smem);
    double *ring_tau = reinterpret_cast<double *>(smem + C::OFF_TAU);
    const uint32_t bar_full = smem_u32(smem + C::OFF_BAR);
    const uint32_t bar_empty = bar_full + NS * 8;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nw = a.nw;
    const int64_t units = (a.nev + C::CW - 1) / C::CW;            // warp-units in the whole call
    const int64_t unit0 = units * blockIdx.x / gridDim.x;           // balanced split over CTAs
    const int64_t nact = units * (blockIdx.x + 1) / gridDim.x - unit0;   // active consumer warps here

    if (threadIdx.x == 0) {
        for (int i = 0; i < NS; ++i) {
            mbar_init(bar_full + 8 * i, 32);
            mbar_init(bar_empty + 8 * i, (uint32_t)nact);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const int64_t N = a.N;
    const int64_t K0 = (N - 2 + NBW) >> C::LG;     // K(0) = ceil((N-1)/nbw): number of chains
    const int64_t B0 = (N - 1) >> 4;

    if (warp == nw) {
        // ================= producer warp: stage reflectors in consumption order =================
        // lane = u + 16*half: reflector u of the block; each half issues LPC/2 of its 16-row groups
        const int u = lane & 15, half = lane >> 4;
        constexpr int GPL = LPC / 2;                          // groups per lane
        constexpr uint32_t GBYTES = 16 * C::ESZ;              // bytes per group
        const int64_t FN1 = hh_F(N - 1, C::LG);
        uint32_t it = 0;
        for (int64_t k = 0; k < K0; ++k) {
            const int64_t Bend = (1 + (k << C::LG)) >> 4;
            for (int64_t B = B0; B >= Bend; --B, ++it) {
                const uint32_t st = it % NS, ph = (it / NS) & 1;
                mbar_wait_backoff(bar_empty + 8 * st, ph ^ 1);
                const int64_t r0 = (B << 4) + u;
                const int64_t s = r0 - 1 - (k << C::LG);
                const bool valid = (r0 <= N - 1) && (s >= 0);
                double tr = 0.0, ti = 0.0;
                int64_t g = 0;
                if (valid) {
                    g = FN1 - hh_F(N - 1 - s, C::LG) + k;
                    tr = __ldg(a.hh_tau + g * EW);
                    if (CPLX) ti = __ldg(a.hh_tau + g * EW + 1);
                }
                if (half == 0) {
                    ring_tau[(st * 16 + u) * EW] = tr;
                    if (CPLX) ring_tau[(st * 16 + u) * EW + 1] = ti;
                }
                if (valid && (tr != 0.0 || ti != 0.0)) {
                    mbar_arrive_expect_tx(bar_full + 8 * st, GPL * GBYTES);
#pragma unroll
                    for (int gg = 0; gg < GPL; ++gg) {
                        const int grp = half * GPL + gg;
                        bulk_g2s(smem_u32(ring_v + ((size_t)(st * 16 + u) * C::VS + grp * C::GS) * EW),
                                 a.hh_v + (g * NBW + grp * 16) * EW, GBYTES, bar_full + 8 * st);
                    }
                } else {
                    mbar_arrive(bar_full + 8 * st);
                }
            }
        }
        return;
    }
    if (warp >= nact) return;

    // ================= consumer warps =================
    const int l = lane % LPC;          // row lane: slots 16l .. 16l+15
    const int cg = lane / LPC;         // column group
    const int64_t col0 = (unit0 + warp) * C::CW;
    double *tiles = reinterpret_cast<double *>(smem + C::OFF_TILE + (size_t)warp * 2 * C::TILE_BYTES);

    double x[CPL][16 * EW];
    uint32_t it = 0;
    for (int64_t k = 0; k < K0; ++k) {
#pragma unroll
        for (int j = 0; j < CPL; ++j)
#pragma unroll
            for (int i = 0; i < 16 * EW; ++i) x[j][i] = 0.0;
        const int64_t Bend = (1 + (k << C::LG)) >> 4;
        tile_fill<C, CPLX>(a, tiles + (B0 & 1) * (C::TILE_BYTES / 8), col0, B0, lane);
        cp_async_commit();
        for (int64_t B = B0; B >= Bend; --B, ++it) {
            cp_async_wait_all();
            __syncwarp();
            if (B > Bend) tile_fill<C, CPLX>(a, tiles + ((B - 1) & 1) * (C::TILE_BYTES / 8), col0, B - 1, lane);
            cp_async_commit();
            const uint32_t st = it % NS, ph = (it / NS) & 1;
            mbar_wait(bar_full + 8 * st, ph);
            const double *vb = ring_v + (size_t)st * 16 * C::VS * EW;
            const double *tb = ring_tau + st * 16 * EW;
            const double *v0 = vb + (((l - (int)B) & (LPC - 1)) * C::GS) * EW;       // slots i >= u
            const double *v1 = vb + (((l - (int)B - 1) & (LPC - 1)) * C::GS) * EW;   // slots i <  u
            const bool act = (l == ((int)B & (LPC - 1)));
            double *tl = tiles + (B & 1) * (C::TILE_BYTES / 8) + cg * C::TSTRIDE * EW;
#pragma unroll
            for (int uu = 0; uu < 16; ++uu) {
                const int u = 15 - uu;
                // --- window turnover: retire row 16B+u+nbw, admit row 16B+u
                if (act) {
#pragma unroll
                    for (int j = 0; j < CPL; ++j) {
                        double *p = tl + (j * NCG * C::TSTRIDE + u) * EW;
                        if (CPLX) {
                            const double2 nw2 = *reinterpret_cast<double2 *>(p);
                            *reinterpret_cast<double2 *>(p) = make_double2(x[j][2 * u], x[j][2 * u + 1]);
                            x[j][2 * u] = nw2.x;
                            x[j][2 * u + 1] = nw2.y;
                        } else {
                            const double nv = *p;
                            *p = x[j][u];
                            x[j][u] = nv;
                        }
                    }
                }
                const double tr = tb[u * EW];
                const double ti = CPLX ? tb[u * EW + 1] : 0.0;
                if (tr != 0.0 || ti != 0.0) {
                    double vv[16 * EW];
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        const double *src = (i >= u) ? v0 + (u * C::VS + (i - u)) * EW
                                                     : v1 + (u * C::VS + (16 + i - u)) * EW;
                        if (CPLX) {
                            const double2 t2 = *reinterpret_cast<const double2 *>(src);
                            vv[2 * i] = t2.x;
                            vv[2 * i + 1] = t2.y;
                        } else {
                            vv[i] = *src;
                        }
                    }
                    // All CPL columns advance together (i outer, column inner): 2*CPL (real) or
                    // 4*CPL (complex) independent FMA chains hide the DFMA latency.
                    if (CPLX) {
                        // d = sum conj(v) x  (R2)
                        double dr[CPL], di[CPL], er[CPL], ei[CPL];
#pragma unroll
                        for (int j = 0; j < CPL; ++j) {
                            dr[j] = vv[0] * x[j][0];
                            er[j] = vv[1] * x[j][1];
                            di[j] = vv[0] * x[j][1];
                            ei[j] = -vv[1] * x[j][0];
                        }
#pragma unroll
                        for (int i = 1; i < 16; ++i)
#pragma unroll
                            for (int j = 0; j < CPL; ++j) {
                                dr[j] = fma(vv[2 * i], x[j][2 * i], dr[j]);
                                er[j] = fma(vv[2 * i + 1], x[j][2 * i + 1], er[j]);
                                di[j] = fma(vv[2 * i], x[j][2 * i + 1], di[j]);
                                ei[j] = fma(-vv[2 * i + 1], x[j][2 * i], ei[j]);
                            }
#pragma unroll
                        for (int j = 0; j < CPL; ++j) {
                            dr[j] += er[j];
                            di[j] += ei[j];
                        }
#pragma unroll
                        for (int m = 1; m < LPC; m <<= 1)
#pragma unroll
                            for (int j = 0; j < CPL; ++j) {
                                dr[j] += shfl_xor_f64(dr[j], m);
                                di[j] += shfl_xor_f64(di[j], m);
                            }
                        double hr[CPL], hi[CPL];   // h = -tau d
#pragma unroll
                        for (int j = 0; j < CPL; ++j) {
                            hr[j] = -(tr * dr[j] - ti * di[j]);
                            hi[j] = -(tr * di[j] + ti * dr[j]);
                        }
#pragma unroll
                        for (int i = 0; i < 16; ++i)
#pragma unroll
                            for (int j = 0; j < CPL; ++j) {
                                double xr = x[j][2 * i], xi = x[j][2 * i + 1];
                                xr = fma(hr[j], vv[2 * i], xr);
                                xi = fma(hr[j], vv[2 * i + 1], xi);
                                xr = fma(-hi[j], vv[2 * i + 1], xr);
                                xi = fma(hi[j], vv[2 * i], xi);
                                x[j][2 * i] = xr;
                                x[j][2 * i + 1] = xi;
                            }
                    } else {
                        // four partial sums per column: even if the scheduler serialises the
                        // columns, four independent chains cover the DFMA latency
                        double d0[CPL], d1[CPL], d2[CPL], d3[CPL];
#pragma unroll
                        for (int j = 0; j < CPL; ++j) {
                            d0[j] = vv[0] * x[j][0];
                            d1[j] = vv[1] * x[j][1];
                            d2[j] = vv[2] * x[j][2];
                            d3[j] = vv[3] * x[j][3];
                        }
#pragma unroll
                        for (int i = 4; i < 16; i += 4)
#pragma unroll
                            for (int j = 0; j < CPL; ++j) {
                                d0[j] = fma(vv[i], x[j][i], d0[j]);
                                d1[j] = fma(vv[i + 1], x[j][i + 1], d1[j]);
                                d2[j] = fma(vv[i + 2], x[j][i + 2], d2[j]);
                                d3[j] = fma(vv[i + 3], x[j][i + 3], d3[j]);
                            }
#pragma unroll
                        for (int j = 0; j < CPL; ++j) d0[j] = (d0[j] + d1[j]) + (d2[j] + d3[j]);
#pragma unroll
                        for (int m = 1; m < LPC; m <<= 1)
#pragma unroll
                            for (int j = 0; j < CPL; ++j) d0[j] += shfl_xor_f64(d0[j], m);
                        double h[CPL];
#pragma unroll
                        for (int j = 0; j < CPL; ++j) h[j] = -tr * d0[j];
#pragma unroll
                        for (int i = 0; i < 16; ++i)
#pragma unroll
                            for (int j = 0; j < CPL; ++j) x[j][i] = fma(h[j], vv[i], x[j][i]);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8 * st);
            tile_drain<C, CPLX>(a, tiles + (B & 1) * (C::TILE_BYTES / 8), col0, B + NBW / 16, lane);
            __syncwarp();
        }
        // --- chain end: the window is rows 16*Bend .. 16*Bend+nbw-1; lane l holds the aligned
        //     16-row block b' = Bend + ((l - Bend) mod LPC) in register order.
        {
            const int64_t rb = (Bend + ((l - (int)Bend) & (LPC - 1))) << 4;
#pragma unroll
            for (int j = 0; j < CPL; ++j) {
                const int64_t col = col0 + cg + j * NCG;
                if (col < a.nev) {
                    double *dst = a.q + (col * a.ldq + rb) * EW;
                    if (CPLX || a.align16) {
#pragma unroll
                        for (int i = 0; i < 16 * EW; i += 2) {
                            const int64_t row = rb + i / EW;
                            if (CPLX ? (row < N) : (row + 1 < N))
                                *reinterpret_cast<double2 *>(dst + i) = make_double2(x[j][i], x[j][i + 1]);
                            else if (!CPLX && row < N)
                                dst[i] = x[j][i];
                        }
                    } else {
#pragma unroll
                        for (int i = 0; i < 16; ++i)
                            if (rb + i < N) dst[i] = x[j][i];
                    }
                }
            }
        }
        __syncwarp();
        __threadfence_block();
    }
}

}  // namespace elpa2bt
