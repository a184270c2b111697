// bt_shift.cuh -- register-resident sliding-window back-transformation kernel (sm_100a).
//
// What it computes: include/elpa2_bt.h (Eq. 6d, Eq. 8).
// How:
//  * Columns of q are independent: a warp owns CW columns for the whole call; CTAs
//    never communicate.
//  * Order: chain-major (k ascending outermost, s descending inside), a dependency-respecting
//    reorder of "reverse generation order" (R5).  Along one chain the
//    nbw-row window moves up by one row per reflector.
//  * The window lives in REGISTERS, indexed by POSITION in the window: x[i] is row r0+i of the
//    reflector being applied, so the v operand of every FMA has a static index and one loop
//    iteration (= one reflector) is the same straight-line code for every reflector.  The shift
//    "up by one row" (PAPER.md:174 step 3) costs nothing: the rank-1 update writes its result one
//    register further down, x[i+1] <- x[i] + h v[i] (an FMA's destination is free to differ from
//    its addend).  A column's nbw rows are split in contiguous pieces of RL rows over LPC lanes;
//    the element that crosses a lane boundary travels by one warp shuffle per step, and the same
//    rotation hands the retired bottom row to lane 0, which swaps it with the admitted top row in
//    the warp's shared-memory tile.
//  * v^H x (PAPER.md:172 step 2a): RL FMAs per lane and column, then log2(LPC) shuffle stages;
//    x <- x - tau d v (PAPER.md:173 step 2b): RL FMAs.  Each lane works on CPL columns, whose
//    dot / reduce / update phases interleave and hide each other's latency.
//  * Reflectors are staged once per CTA by a producer warp with 1-D bulk copies (TMA engine,
//    UBLKCP) into a ring of 16-reflector blocks guarded by full/empty mbarriers.
//  * Rows enter/leave through per-warp 16-row tiles: cp.async fill of the 16 rows above the
//    window (one full 128-byte line per column), in-place exchange new<->retired during the 16
//    steps, coalesced 16-byte stores of the retired rows.
#pragma once
#include "bt_common.cuh"

namespace elpa2bt {

template <bool CPLX, int NBW_, int CPL_>
struct ShiftCfg {
    static constexpr int NBW = NBW_;
    static constexpr int LG = (NBW == 32) ? 5 : (NBW == 64) ? 6 : 7;
    static constexpr int CPL = CPL_;                 // columns per lane
    static constexpr int EW = CPLX ? 2 : 1;          // doubles per element
    static constexpr int ESZ = 8 * EW;
    static constexpr int RL = CPLX ? 16 : 32;        // window rows per lane
    static constexpr int LPC = NBW / RL;             // lanes sharing one column
    static constexpr int NCG = 32 / LPC;             // column groups per warp
    static constexpr int CW = NCG * CPL;             // columns per warp
    static constexpr int TSTRIDE = CPLX ? 17 : 18;   // tile column stride (elements), 16-byte aligned
    static constexpr int TILE_BYTES = CW * TSTRIDE * ESZ;
    // v in shared memory: LPC groups of RL rows, group stride padded by 16 bytes so that the LPC
    // row lanes of a column (same offset, different groups) read from different banks
    static constexpr int GS = RL + (CPLX ? 1 : 2);    // group stride (elements)
    static constexpr int VS = LPC * GS;               // reflector stride (elements)
    static constexpr int VBLK_BYTES = 16 * VS * ESZ;
    static constexpr int TAU_BYTES = 16 * ESZ;
    static constexpr int NS = 4;                      // ring stages
    static constexpr int OFF_TAU = NS * VBLK_BYTES;
    static constexpr int OFF_BAR = OFF_TAU + NS * TAU_BYTES;
    static constexpr int OFF_TILE = OFF_BAR + 2 * NS * 8;
    static_assert(OFF_TILE % 16 == 0, "tile alignment");
    static_assert((GS * ESZ) % 16 == 0, "v group alignment");
    static size_t smem_bytes(int nw) { return (size_t)OFF_TILE + (size_t)nw * 2 * TILE_BYTES; }
};

// ---- tile fill / drain -------------------------------------------------------------------------
// Tile buffer: element (c, r) of the warp's CW x 16 block at tile[(c*TSTRIDE + r) * EW].
template <class C, bool CPLX>
__device__ __forceinline__ void sh_tile_fill(const WinArgs &a, double *tile, int64_t col0, int64_t B, int lane)
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
__device__ __forceinline__ void sh_tile_drain(const WinArgs &a, const double *tile, int64_t col0, int64_t Bout, int lane)
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

// ---- one reflector on the CPL columns of a lane ------------------------------------------------
// x[j][i]: window position p*RL + i of column j (position 0 = row r0 of the reflector); on entry
// x[j][0] is free and c[j] holds what left the lane's piece in the previous step.  vb: this lane's
// RL-row piece of v in the ring; (tr, ti) = tau; slot: tile element (column 0 of the lane, row r0).
template <class C, bool CPLX>
__device__ __forceinline__ void reflector_step(double (&x)[C::CPL][C::RL * C::EW], double (&c)[C::CPL][C::EW],
                                               const double *__restrict__ vb, const double tr, const double ti,
                                               double *slot, const int p, const int src_lane)
{
    constexpr int CPL = C::CPL, RL = C::RL, EW = C::EW, LPC = C::LPC;
    // --- window turnover (PAPER.md:174 step 3): the element that left lane p-1 enters lane p;
    //     lane 0 gets the retired bottom row from lane LPC-1 and swaps it with the admitted row
#pragma unroll
    for (int j = 0; j < CPL; ++j) {
        double t0 = c[j][0], t1 = CPLX ? c[j][EW - 1] : 0.0;
        if (LPC > 1) {
            t0 = __shfl_sync(0xffffffffu, t0, src_lane);
            if (CPLX) t1 = __shfl_sync(0xffffffffu, t1, src_lane);
        }
        if (p == 0) {
            double *e = slot + j * C::NCG * C::TSTRIDE * EW;
            if (CPLX) {
                const double2 nw2 = *reinterpret_cast<double2 *>(e);
                *reinterpret_cast<double2 *>(e) = make_double2(t0, t1);
                t0 = nw2.x;
                t1 = nw2.y;
            } else {
                const double nv = *e;
                *e = t0;
                t0 = nv;
            }
        }
        x[j][0] = t0;
        if (CPLX) x[j][EW - 1] = t1;
    }
    // --- this lane's piece of v
    double vv[RL * EW];
#pragma unroll
    for (int i = 0; i < RL * EW; i += 2) {
        const double2 t2 = *reinterpret_cast<const double2 *>(vb + i);
        vv[i] = t2.x;
        vv[i + 1] = t2.y;
    }
    if (CPLX) {
        double hr[CPL], hi[CPL];
#pragma unroll
        for (int j = 0; j < CPL; ++j) {
            // d = sum conj(v) x  (PAPER.md:172 step 2a; R2); position 0 last: it arrives latest
            double dr = vv[2] * x[j][2], er = vv[3] * x[j][3], di = vv[2] * x[j][3], ei = -vv[3] * x[j][2];
#pragma unroll
            for (int i = 2; i < RL; ++i) {
                dr = fma(vv[2 * i], x[j][2 * i], dr);
                er = fma(vv[2 * i + 1], x[j][2 * i + 1], er);
                di = fma(vv[2 * i], x[j][2 * i + 1], di);
                ei = fma(-vv[2 * i + 1], x[j][2 * i], ei);
            }
            dr = fma(vv[0], x[j][0], dr);
            er = fma(vv[1], x[j][1], er);
            di = fma(vv[0], x[j][1], di);
            ei = fma(-vv[1], x[j][0], ei);
            dr += er;
            di += ei;
#pragma unroll
            for (int m = 1; m < LPC; m <<= 1) {
                dr += __shfl_xor_sync(0xffffffffu, dr, m);
                di += __shfl_xor_sync(0xffffffffu, di, m);
            }
            hr[j] = -(tr * dr - ti * di);      // h = -tau d
            hi[j] = -(tr * di + ti * dr);
        }
#pragma unroll
        for (int j = 0; j < CPL; ++j) {
            // x <- x + h v, written one position further down (PAPER.md:173 step 2b + :174 step 3)
            {
                double xr = x[j][2 * RL - 2], xi = x[j][2 * RL - 1];
                xr = fma(hr[j], vv[2 * RL - 2], xr);
                xi = fma(hr[j], vv[2 * RL - 1], xi);
                xr = fma(-hi[j], vv[2 * RL - 1], xr);
                xi = fma(hi[j], vv[2 * RL - 2], xi);
                c[j][0] = xr;
                c[j][1] = xi;
            }
#pragma unroll
            for (int i = RL - 2; i >= 0; --i) {
                double xr = x[j][2 * i], xi = x[j][2 * i + 1];
                xr = fma(hr[j], vv[2 * i], xr);
                xi = fma(hr[j], vv[2 * i + 1], xi);
                xr = fma(-hi[j], vv[2 * i + 1], xr);
                xi = fma(hi[j], vv[2 * i], xi);
                x[j][2 * i + 2] = xr;
                x[j][2 * i + 3] = xi;
            }
        }
    } else {
        double h[CPL];
#pragma unroll
        for (int j = 0; j < CPL; ++j) {
            double d0 = vv[1] * x[j][1], d1 = vv[2] * x[j][2], d2 = vv[3] * x[j][3], d3 = vv[4] * x[j][4];
#pragma unroll
            for (int i = 5; i + 3 < RL; i += 4) {
                d0 = fma(vv[i], x[j][i], d0);
                d1 = fma(vv[i + 1], x[j][i + 1], d1);
                d2 = fma(vv[i + 2], x[j][i + 2], d2);
                d3 = fma(vv[i + 3], x[j][i + 3], d3);
            }
            // RL = 32: i stops at 29; positions 29, 30, 31 and 0 remain
            d0 = fma(vv[RL - 3], x[j][RL - 3], d0);
            d1 = fma(vv[RL - 2], x[j][RL - 2], d1);
            d2 = fma(vv[RL - 1], x[j][RL - 1], d2);
            d3 = fma(vv[0], x[j][0], d3);
            double d = (d0 + d1) + (d2 + d3);
#pragma unroll
            for (int m = 1; m < LPC; m <<= 1) d += __shfl_xor_sync(0xffffffffu, d, m);
            h[j] = -tr * d;
        }
#pragma unroll
        for (int j = 0; j < CPL; ++j) {
            c[j][0] = fma(h[j], vv[RL - 1], x[j][RL - 1]);
#pragma unroll
            for (int i = RL - 2; i >= 0; --i) x[j][i + 1] = fma(h[j], vv[i], x[j][i]);
        }
    }
}

// ---- the kernel -------------------------------------------------------------------------------
template <bool CPLX, int NBW, int CPL, int MAXT, int UNROLL>
__global__ void __launch_bounds__(MAXT, 1) bt_shift_kernel(const WinArgs a)
{
    using C = ShiftCfg<CPLX, NBW, CPL>;
    constexpr int EW = C::EW, LPC = C::LPC, NCG = C::NCG, NS = C::NS, RL = C::RL;
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

    // the ring starts as zeros: slots outside a chain's range are never copied and their (stale
    // or initial) v is multiplied by h = -0 * d, which must stay finite
    for (int i = threadIdx.x; i < C::OFF_BAR / 8; i += blockDim.x) ring_v[i] = 0.0;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (threadIdx.x == 0) {
        for (int i = 0; i < NS; ++i) {
            mbar_init(bar_full + 8 * i, 32);
            mbar_init(bar_empty + 8 * i, (uint32_t)nact);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const int64_t N = a.N;
    const int64_t K0 = (N - 2 + NBW) / NBW;     // K(0) = ceil((N-1)/nbw): number of chains
    const int64_t B0 = (N - 1) >> 4;

    if (warp == nw) {
        // ================= producer warp: stage reflectors in consumption order =================
        // a block = 16 reflectors x LPC pieces of RL rows; copy id = lane + 32 t -> (u, piece)
        constexpr int NCOPY = 16 * LPC;
        constexpr int CPLN = (NCOPY + 31) / 32;               // copies per lane
        constexpr uint32_t PBYTES = RL * C::ESZ;              // bytes per piece
        const int u = lane & 15;
        const int64_t FN1 = hh_F(N - 1, NBW);
        uint32_t it = 0;
        for (int64_t k = 0; k < K0; ++k) {
            const int64_t Bend = (1 + (k * NBW)) >> 4;
            for (int64_t B = B0; B >= Bend; --B, ++it) {
                const uint32_t st = it % NS, ph = (it / NS) & 1;
                mbar_wait_backoff(bar_empty + 8 * st, ph ^ 1);
                const int64_t r0 = (B << 4) + u;
                const int64_t s = r0 - 1 - (k * NBW);
                const bool valid = (r0 <= N - 1) && (s >= 0);
                double tr = 0.0, ti = 0.0;
                int64_t g = 0;
                if (valid) {
                    g = FN1 - hh_F(N - 1 - s, NBW) + k;
                    tr = __ldg(a.hh_tau + g * EW);
                    if (CPLX) ti = __ldg(a.hh_tau + g * EW + 1);
                }
                if (lane < 16) {
                    ring_tau[(st * 16 + u) * EW] = tr;
                    if (CPLX) ring_tau[(st * 16 + u) * EW + 1] = ti;
                }
                const bool mine = valid && (lane < NCOPY);
                if (mine) {
                    constexpr int NMINE = (NCOPY >= 32) ? CPLN : 1;
                    mbar_arrive_expect_tx(bar_full + 8 * st, NMINE * PBYTES);
#pragma unroll
                    for (int t = 0; t < NMINE; ++t) {
                        const int piece = (lane >> 4) + 2 * t;
                        bulk_g2s(smem_u32(ring_v + ((size_t)(st * 16 + u) * C::VS + piece * C::GS) * EW),
                                 a.hh_v + (g * NBW + piece * RL) * EW, PBYTES, bar_full + 8 * st);
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
    const int p = lane % LPC;          // row lane: window positions p*RL .. p*RL+RL-1
    const int cg = lane / LPC;         // column group: columns cg + NCG*j
    const int src_lane = (lane - p) + ((p + LPC - 1) % LPC);
    const int64_t col0 = (unit0 + warp) * C::CW;
    double *tiles = reinterpret_cast<double *>(smem + C::OFF_TILE + (size_t)warp * 2 * C::TILE_BYTES);

    double x[CPL][RL * EW];
    double c[CPL][EW];
    uint32_t it = 0;
    for (int64_t k = 0; k < K0; ++k) {
#pragma unroll
        for (int j = 0; j < CPL; ++j) {
#pragma unroll
            for (int i = 0; i < RL * EW; ++i) x[j][i] = 0.0;
#pragma unroll
            for (int i = 0; i < EW; ++i) c[j][i] = 0.0;
        }
        const int64_t Bend = (1 + (k * NBW)) >> 4;
        sh_tile_fill<C, CPLX>(a, tiles + (B0 & 1) * (C::TILE_BYTES / 8), col0, B0, lane);
        cp_async_commit();
        for (int64_t B = B0; B >= Bend; --B, ++it) {
            cp_async_wait_all();
            __syncwarp();
            if (B > Bend) sh_tile_fill<C, CPLX>(a, tiles + ((B - 1) & 1) * (C::TILE_BYTES / 8), col0, B - 1, lane);
            cp_async_commit();
            const uint32_t st = it % NS, ph = (it / NS) & 1;
            mbar_wait(bar_full + 8 * st, ph);
            const double *vb = ring_v + ((size_t)st * 16 * C::VS + p * C::GS) * EW;
            const double *tb = ring_tau + st * 16 * EW;
            double *tl = tiles + (B & 1) * (C::TILE_BYTES / 8) + cg * C::TSTRIDE * EW;
#pragma unroll UNROLL
            for (int u = 15; u >= 0; --u) {
                const double tr = tb[u * EW];
                const double ti = CPLX ? tb[u * EW + 1] : 0.0;
                reflector_step<C, CPLX>(x, c, vb + u * C::VS * EW, tr, ti, tl + u * EW, p, src_lane);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8 * st);
            sh_tile_drain<C, CPLX>(a, tiles + (B & 1) * (C::TILE_BYTES / 8), col0, B + NBW / 16, lane);
            __syncwarp();
        }
        // --- chain end: lane p holds rows 16*Bend + p*RL + (0 .. RL-1) as x[1..RL-1], c
        {
            const int64_t rb = (Bend << 4) + p * RL;
#pragma unroll
            for (int j = 0; j < CPL; ++j) {
                const int64_t col = col0 + cg + j * NCG;
                if (col < a.nev) {
                    double *dst = a.q + (col * a.ldq + rb) * EW;
                    if (CPLX) {
#pragma unroll
                        for (int i = 0; i < RL; ++i) {
                            const double vr = (i < RL - 1) ? x[j][2 * i + 2] : c[j][0];
                            const double vi = (i < RL - 1) ? x[j][2 * i + 3] : c[j][1];
                            if (rb + i < N) *reinterpret_cast<double2 *>(dst + 2 * i) = make_double2(vr, vi);
                        }
                    } else if (a.align16) {
#pragma unroll
                        for (int i = 0; i < RL; i += 2) {
                            const double v0 = x[j][i + 1];
                            const double v1 = (i + 1 < RL - 1) ? x[j][i + 2] : c[j][0];
                            if (rb + i + 1 < N)
                                *reinterpret_cast<double2 *>(dst + i) = make_double2(v0, v1);
                            else if (rb + i < N)
                                dst[i] = v0;
                        }
                    } else {
#pragma unroll
                        for (int i = 0; i < RL; ++i) {
                            const double v0 = (i < RL - 1) ? x[j][i + 1] : c[j][0];
                            if (rb + i < N) dst[i] = v0;
                        }
                    }
                }
            }
        }
        __syncwarp();
        __threadfence_block();
    }
}

}  // namespace elpa2bt
