// bt_wy.cuh -- compact-WY back-transformation on the FP64 tensor cores (DMMA m8n8k4), real FP64,
// sm_100a.  What it computes: include/elpa2_bt.h (Eq. 6d, Eq. 8).
//
// M = 8 consecutive reflectors of a chain (first rows r0 = 8b+7, 8b+6, .., 8b: applied in that
// order) are aggregated (R6; PAPER.md:54, :101 cite the technique):
//      H_7 .. H_1 H_0 = I - V T V^T,   T lower triangular, T[j][j] = tau_j,
//      T[j][:j] = -tau_j (v_j^T V[:, :j]) T[:j, :j],
// where V is the W x 8 matrix (W = nbw + 8 window rows 8b .. 8b+W-1) whose column i holds v_i at
// row offset 7 - i.  With Y = V (-T) (W x 8, computed once per block by wy_prepass_kernel) the
// window x (W x 8 per slab of 8 columns) is updated by
//      D^T = x^T V        (8 cols x 8 refl, K = W rows)       W/4  DMMAs
//      x^T += D^T Y^T     (8 cols x W rows, K = 8)            W/4  DMMAs
// i.e. (nbw/2 + 4) DMMAs for the nbw/2 DMMA-equivalents of useful work (4 L flops per reflector
// and column): 89 % at nbw = 64.  Both products keep "column of q" on the M index of the fragment
// (lane / 4) and permute the K index so that the C fragment of the first product IS the A fragment
// of the second: no shuffles, no shared-memory round trip for x or D.
//
//  * x^T fragment: lane (gq = lane/4, r = lane%4) holds rows 8t + 2r + {0,1} of column gq for
//    every 8-row tile t of the window: NT = W/8 register pairs per slab.  This is the C layout of
//    the update (M = column, N = row in tile) and, read as "k-slot r of k-chunk (t,e) is row
//    8t + 2r + e", the A layout of the dot product.
//  * The window moves up by 8 rows = one tile per block: the update of tile t writes its result
//    into the registers of tile t+1 (D != C in the DMMA), tile NT-1 retires to global memory
//    (16 bytes per lane, 64 contiguous bytes per column), tile 0 is loaded one or two blocks ahead.
//  * Shared memory per block: VA[i][w] = V (B fragments of the dot product), staged by 8-byte
//    cp.async straight from hh_v (the skew 7 - i breaks the 16-byte alignment bulk copies need), and
//    YB[w][j] = Y (B fragments of the update), one bulk copy (TMA engine) of the image the prepass
//    left in the scratch array.
//  * 8 warps per CTA (2 per SM sub-partition, 255 registers), no producer warp: the warps take
//    turns at staging block it+NS-LAG; completion is tracked on the stage's full mbarrier by
//    cp.async.mbarrier.arrive and the bulk copy's byte count.
//  * Few columns: chain-parallel mode (P warps per slab on interleaved chains, see prog_publish).
//  * Order across chains: chain-major (R5), as in the other kernels.
#pragma once
#include "bt_common.cuh"

namespace elpa2bt {

template <int NBW_, int NW_ = 8>
struct WyCfg {
    static constexpr int NBW = NBW_;                  // any multiple of 16 (R13: the library instantiates multiples of 32)
    static constexpr int NB8 = NBW / 8;               // 8-row blocks per chase block
    static constexpr int NT = NBW / 8 + 1;            // 8-row tiles in the window
    static constexpr int W = 8 * NT;                  // window rows (= nbw + 8; W % 16 == 8)
    static constexpr int NW = NW_;                    // warps per CTA: 8 (255 registers) or, for few columns, 16 (128)
    static constexpr int NGMAX = (NW_ > 8) ? 1 : (NBW <= 64) ? 4 : (NBW <= 128) ? 2 : 1;   // most 8-column slabs per warp
    // ring stages: 8 (16 in the 16-warp build) while 8 stages of 16 W doubles fit, else 4
    static constexpr int NS = (NW_ > 8) ? 16 : (8 * 16 * W * 8 <= 216 * 1024) ? 8 : 4;
    static constexpr int LGNS = (NS == 16) ? 4 : (NS == 8) ? 3 : 2;
    static constexpr int LAG = 4;                     // staging waits for the block LAG iterations back
    static constexpr int VA_OFF = 0;                  // VA[i][w] = V, row stride W
    static constexpr int YB_OFF = 8 * W;              // YB[w][j] = (V (-T))[w][j], row stride 8
    static constexpr int STAGE_DOUBLES = 16 * W;
    static constexpr int YBLK = 8 * W;                // doubles of scratch per block (its YB image)
    static constexpr int PW = (NBW <= 64) ? 8 : (NBW <= 128) ? 4 : 2;    // warps (= blocks) per CTA of the prepass kernel
    static constexpr int OFF_BAR = NS * STAGE_DOUBLES * 8;
    static constexpr int SMEM_BYTES = OFF_BAR + 2 * NS * 8;
    static_assert(W % 16 == 8, "VA row stride must be 8 mod 16 doubles (bank-conflict-free LDS.128)");
    static_assert(SMEM_BYTES <= 227 * 1024, "shared memory");
};

struct WyArgs {
    int64_t N, nev, ldq;
    const double *hh_v;    // G * nbw
    const double *hh_tau;  // G
    double *q;
    double *tn;            // scratch of the prepass, per block in consumption order (real: the YB image)
    uint32_t *prog;        // chain-parallel mode: prog[slab * K0 + k] = blocks of chain k finished (zeroed per call)
    int align16;           // q base and ldq*8 are 16-byte aligned
    int P;                 // warps per slab (1, 2 or 4), each on its own chains k = p, p+P, ...
    // Sub-range launches (rowpipe: a rank that owns a block of rows): chains [kb, ke),
    // of each chain only the blocks b_bot <= b <= b_top; rows >= row_end are not in memory (read as zero,
    // never written); q and tn are pre-shifted so that global row / block indices address them.  The whole
    // matrix is kb = 0, ke = K0, b_top = bhi, b_bot = 0, row_end = N.
    int64_t kb, ke, b_top, b_bot, row_end;
};

// ---- block enumeration ----------------------------------------------------------------------------
// chain k = 0 .. K0-1 (K0 = ceil((N-1)/nbw)); within a chain, blocks b = bhi down to k*nbw/8, where
// bhi = (N-1)/8.  id(k, b) = base(k) + (bhi - b) is the consumption order.
__host__ __device__ __forceinline__ int64_t wy_bhi(int64_t N) { return (N - 1) >> 3; }
__host__ __device__ __forceinline__ int64_t wy_base(int64_t N, int nbw, int64_t k)
{
    return k * (wy_bhi(N) + 1) - (int64_t)(nbw >> 3) * ((k * (k - 1)) >> 1);
}
__host__ __device__ __forceinline__ int64_t wy_nchains(int64_t N, int nbw) { return (N - 2 + nbw) / nbw; }
__host__ __device__ __forceinline__ int64_t wy_nblocks(int64_t N, int nbw) { return wy_base(N, nbw, wy_nchains(N, nbw)); }

// slot of reflector i of block (k, b) (first row r0 = 8b + 7 - i; sweep s = r0 - 1 - k nbw; R3),
// -1 if the block position is outside the chain
template <int NBW>
__device__ __forceinline__ int64_t wy_slot(int64_t N, int64_t FN1, int64_t k, int64_t b, int i)
{
    const int64_t r0 = (b << 3) + 7 - i;
    const int64_t s = r0 - 1 - k * NBW;
    if (r0 > N - 1 || s < 0) return -1;
    return FN1 - hh_F(N - 1 - s, NBW) + k;
}

__device__ __forceinline__ void dmma884(double &d0, double &d1, const double a, const double b, const double c0,
                                        const double c1)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%4,%5};"
        : "=d"(d0), "=d"(d1)
        : "d"(a), "d"(b), "d"(c0), "d"(c1));
}

__device__ __forceinline__ void cp_async_mbar_arrive_noinc_wy(uint32_t bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}

// ---- prepass: Y = V (-T) of every block ------------------------------------------------------------
// grid (ceil((bhi+1)/PW), K0), PW warps: warp = one block (k, b).  Lane (gq, r) loads column gq
// of V at window rows 4c + r, c = 0 .. W/4-1 (both the A and the B fragment of V^T V; also parked in
// shared memory), the Gram matrix comes out of W/4 DMMAs, lane l & 7 runs the recurrence of R6 for
// column l of T, and W/4 more DMMAs give Y = V (-T), stored as the YB[w][j] image the main kernel
// stages with one bulk copy.
template <int NBW>
__global__ void __launch_bounds__(WyCfg<NBW>::PW * 32) wy_prepass_kernel(int64_t N, const double *__restrict__ hh_v,
                                                                         const double *__restrict__ hh_tau,
                                                                         double *__restrict__ yb, int64_t kb)
{
    using C = WyCfg<NBW>;
    constexpr int W = C::W, SV = W + 2;               // Vs row stride: rows r, r+1 land 4 banks apart
    __shared__ double Sm[C::PW][64];
    __shared__ double Vs[C::PW][8 * SV];
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
    const double tau = slot >= 0 ? hh_tau[slot] : 0.0;
    double s0 = 0.0, s1 = 0.0, u0 = 0.0, u1 = 0.0;
#pragma unroll
    for (int c = 0; c < W / 4; ++c) {
        const int rl = 4 * c + r - (7 - gq);
        const double v = (slot >= 0 && rl >= 0 && rl < NBW) ? hh_v[slot * NBW + rl] : 0.0;
        Vs[warp][gq * SV + 4 * c + r] = v;
        if (c & 1)
            dmma884(u0, u1, v, v, u0, u1);
        else
            dmma884(s0, s1, v, v, s0, s1);
    }
    // S[m = gq][n = 2r + {0,1}]
    Sm[warp][gq * 8 + 2 * r] = s0 + u0;
    Sm[warp][gq * 8 + 2 * r + 1] = s1 + u1;
    __syncwarp();
    const int l = lane & 7;
    double t[8];
#pragma unroll
    for (int jj = 0; jj < 8; ++jj) {
        const double tau_j = __shfl_sync(0xffffffffu, tau, 4 * jj);
        double acc = 0.0;
#pragma unroll
        for (int i = 0; i < jj; ++i) acc = fma(Sm[warp][jj * 8 + i], t[i], acc);
        t[jj] = (jj == l) ? tau_j : (jj > l ? -tau_j * acc : 0.0);
    }
    __syncwarp();
    if (lane < 8) {
#pragma unroll
        for (int jj = 0; jj < 8; ++jj) Sm[warp][jj * 8 + l] = -t[jj];      // Sm = -T, row-major [i][j]
    }
    __syncwarp();
    // Y[w][j] = sum_i V[w][i] (-T)[i][j]: M = rows of a tile, N = j, K = i (two k-chunks)
    const double tb0 = Sm[warp][r * 8 + gq], tb1 = Sm[warp][(r + 4) * 8 + gq];
    double *out = yb + (wy_base(N, C::NBW, k) + j) * C::YBLK;
#pragma unroll
    for (int tt = 0; tt < C::NT; ++tt) {
        double y0 = 0.0, y1 = 0.0;
        dmma884(y0, y1, Vs[warp][r * SV + 8 * tt + gq], tb0, y0, y1);
        dmma884(y0, y1, Vs[warp][(r + 4) * SV + 8 * tt + gq], tb1, y0, y1);
        *reinterpret_cast<double2 *>(out + (8 * tt + gq) * 8 + 2 * r) = make_double2(y0, y1);
    }
}

// ---- staging one block (whole warp) -----------------------------------------------------------------
// full barrier: 32 cp.async arrivals (one per lane) + 1 arrival carrying the bulk copy's byte count
template <class C>
__device__ __forceinline__ void wy_stage(const WyArgs &a, double *stage, uint32_t bar_full, int64_t k, int64_t b,
                                         int64_t id, int64_t FN1, int lane)
{
    constexpr int NBW = C::NBW, W = C::W;
    const int i8 = lane & 7;
    const int64_t slot = wy_slot<C::NBW>(a.N, FN1, k, b, i8);
    // YB: the prepass wrote the shared-memory image; one bulk copy (TMA engine)
    if (lane == 0) {
        mbar_arrive_expect_tx(bar_full, C::YBLK * 8u);
        bulk_g2s(smem_u32(stage + C::YB_OFF), a.tn + id * C::YBLK, C::YBLK * 8u, bar_full);
    }
    // VA[i][7 - i + r]: lanes run along r (256 contiguous bytes of hh_v per instruction); the skew
    // 7 - i breaks the 16-byte alignment a bulk copy needs, hence 8-byte cp.async
#pragma unroll
    for (int t = 0; t < 8 * NBW / 32; ++t) {
        const int i = (t * 32) / NBW;
        const int rr = (t * 32) % NBW + lane;
        const int64_t sl = __shfl_sync(0xffffffffu, slot, i);
        if (sl >= 0) cp_async8(smem_u32(stage + C::VA_OFF + i * W + 7 - i + rr), a.hh_v + sl * NBW + rr, 8u);
    }
    cp_async_mbar_arrive_noinc_wy(bar_full);
}

// ---- chain-parallel hand-over (P > 1) ------------------------------------------------------------------
// Chain k+1 may load tile 0 of its block b once chain k has retired rows 8b .. 8b+7, i.e. finished
// block b - nbw/8 (R5: chain k+1 needs only what chain k has made final).  The writer publishes
// "blocks finished" with a release store after its tile stores; the reader polls with acquire loads.
// All warps of a slab sit in one CTA, so CTA scope is enough (at GPU scope the release compiles to
// MEMBAR.GPU + ERRBAR and costs 27 % of the kernel); q is still read with ld.global.cg.
__device__ __forceinline__ void prog_publish(uint32_t *p, uint32_t v)
{
    asm volatile("st.release.cta.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t prog_read(const uint32_t *p)
{
    uint32_t v;
    asm volatile("ld.acquire.cta.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// ---- tile I/O: rows row0 + 2r + {0,1} of this lane's column ------------------------------------------
template <bool CG = false>
__device__ __forceinline__ void wy_load2(const WyArgs &a, const int64_t nrow, const double *colp, bool colok, int64_t row,
                                         double &x0, double &x1)
{
    x0 = 0.0;
    x1 = 0.0;
    if (!colok || row >= nrow) return;
    if (a.align16 && row + 1 < nrow) {
        const double2 v = CG ? __ldcg(reinterpret_cast<const double2 *>(colp + row))
                             : *reinterpret_cast<const double2 *>(colp + row);
        x0 = v.x;
        x1 = v.y;
    } else {
        x0 = CG ? __ldcg(colp + row) : colp[row];
        if (row + 1 < nrow) x1 = CG ? __ldcg(colp + row + 1) : colp[row + 1];
    }
}
__device__ __forceinline__ void wy_store2(const WyArgs &a, const int64_t nrow, double *colp, bool colok, int64_t row, double x0,
                                          double x1)
{
    if (!colok || row >= nrow) return;
    if (a.align16 && row + 1 < nrow) {
        *reinterpret_cast<double2 *>(colp + row) = make_double2(x0, x1);
    } else {
        colp[row] = x0;
        if (row + 1 < nrow) colp[row + 1] = x1;
    }
}

// ---- a warp with NG slabs of 8 columns ---------------------------------------------------------------
// CP = false: the 8 warps of a CTA share one ring and walk every chain (grp = 0, member = warp).
// CP = true: a.P warps share NG slabs; warp (grp, member) walks chains grp, grp+P, .. of the slabs
// starting at `slab`; the warps with the same grp share ring grp (NS/P stages) and are its `nmem` members.
template <class C, int NG, bool CP, bool RG>
__device__ __forceinline__ void wy_consume(const WyArgs &a, unsigned char *smem, const int lane, const int grp,
                                           const int member, const int nmem, const int64_t col0, const int64_t slab)
{
    constexpr int NT = C::NT, W = C::W, NBW = C::NBW;
    constexpr int NACC = (NG >= 3) ? 1 : 2;          // dot-product accumulator sets per slab
    const int P = CP ? a.P : 1;
    const int lgs = CP ? (P == 2 ? C::LGNS - 1 : C::LGNS - 2) : C::LGNS;   // log2(stages of this ring), P <= 4
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
    const int64_t kb = RG ? a.kb : 0, ke = RG ? a.ke : K0;
    const int64_t FN1 = hh_F(N - 1, C::NBW);

    // this lane's columns: col0 + 8g + gq, g = 0 .. NG-1
    double *const cb = a.q + (col0 + gq < a.nev ? col0 + gq : 0) * a.ldq;
    const int64_t ldq8 = a.ldq << 3;
    const int64_t ncolrem = a.nev - col0 - gq;          // column g is valid iff 8g < ncolrem
    // warp-uniform fast path of the tile I/O: every column of the warp exists and 16-byte accesses
    // are allowed; then only the first blocks of a chain (rows beyond N) need the guarded code
    const bool fastio = a.align16 && (col0 + 8 * NG <= a.nev);

    // staging cursor: block it + NSP - LAG of this ring's sequence
    auto bbot = [&](int64_t k) { return (RG && k * C::NB8 < a.b_bot) ? a.b_bot : k * C::NB8; };   // last block of chain k here
    int64_t pk = kb + grp, pb = btop;
    auto advance = [&]() {
        if (pb > bbot(pk)) {
            --pb;
        } else {
            pk += P;
            pb = btop;
        }
    };
    auto stage_cursor = [&](uint32_t st) {
        wy_stage<C>(a, ring + st * C::STAGE_DOUBLES, bar_full + 8 * st, pk, pb, wy_base(N, C::NBW, pk) + (bhi - pb), FN1,
                    lane);
    };
    // prologue: blocks 0 .. NSP-LAG-1 go into fresh stages
    for (int i = 0; i < NSP - LAG; ++i) {
        if (member == 0 && pk < ke) stage_cursor((uint32_t)i);
        advance();
    }

    // tile 0 is loaded one block ahead of its block; two blocks ahead when a warp has so few slabs
    // that a block is shorter than a DRAM round trip (Pf holds the tile of the block after next)
    constexpr bool PF2 = (NG <= 2);
    // X[g][t], t = 1 .. NT-1: tiles of the window above tile 0; X[g][NT]: the tile that retires.
    // Tile 0 lives in TA / TB: with PF2 the blocks alternate between the two buffers (a buffer is
    // refilled with the tile of the block after next as soon as its block is done, so no register
    // copy ever waits for a load); otherwise every block uses TA.
    double X[NG][NT + 1][2], TA[NG][2], TB[NG][2];
    uint32_t it = 0;                   // blocks consumed from this ring
    int duty = 0;
    for (int64_t k = kb + grp; k < ke; k += P) {
        const int64_t blo = bbot(k);
        // chain-parallel hand-over: chain k-1 of this slab is walked by another warp of the CTA
        const uint32_t *prev = (CP && k > kb) ? a.prog + slab * K0 + (k - 1) : nullptr;
        uint32_t *mine = CP ? a.prog + slab * K0 + k : nullptr;
        uint32_t known = 0;
        auto wait_prev = [&](int64_t b) {          // before loading tile 0 of block b
            if (CP && prev) {
                const uint32_t need = (uint32_t)(btop - b + NBW / 8 + 1);
                while (known < need) known = prog_read(prev);
            }
        };
        auto load_tile0 = [&](int64_t b, double (&T0)[NG][2]) {
            if (b < blo) return;
            wait_prev(b);
#pragma unroll
            for (int g = 0; g < NG; ++g)
                wy_load2<CP>(a, nrow, cb + g * ldq8, 8 * g < ncolrem, (b << 3) + 2 * r, T0[g][0], T0[g][1]);
        };
        // one block: T0 = its tile 0 on entry, tile 0 of block b - (PF2 ? 2 : 1) on exit
        auto do_block = [&](const int64_t b, double (&T0)[NG][2]) {
            // --- staging duty: block it+NSP-LAG goes into the stage that block it-LAG used; the warp
            //     on duty only waits if some member is still LAG blocks behind it
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
            const double *va = stage + C::VA_OFF + gq * W + 2 * r;
            const double *vb = stage + C::YB_OFF + gq * 8 + 2 * r;

            // --- D^T = x^T V: k-chunk (t, e) = rows 8t + 2r' + e; tile 0 (loaded last) goes last
            double D[NG][NACC][2];
#pragma unroll
            for (int g = 0; g < NG; ++g)
#pragma unroll
                for (int s = 0; s < NACC; ++s) D[g][s][0] = D[g][s][1] = 0.0;
#pragma unroll
            for (int tt = 0; tt < NT; ++tt) {
                const int t = (tt + 1) % NT;
                const double2 v2 = *reinterpret_cast<const double2 *>(va + 8 * t);
#pragma unroll
                for (int g = 0; g < NG; ++g)
                    dmma884(D[g][0][0], D[g][0][1], t ? X[g][t][0] : T0[g][0], v2.x, D[g][0][0], D[g][0][1]);
#pragma unroll
                for (int g = 0; g < NG; ++g)
                    dmma884(D[g][NACC - 1][0], D[g][NACC - 1][1], t ? X[g][t][1] : T0[g][1], v2.y, D[g][NACC - 1][0],
                            D[g][NACC - 1][1]);
            }
            // --- E^T = D^T: T is folded into YB = V (-T), so the dot product feeds the update directly
            double E[NG][2];
#pragma unroll
            for (int g = 0; g < NG; ++g) {
                E[g][0] = D[g][0][0];
                E[g][1] = D[g][0][1];
                if (NACC == 2) {
                    E[g][0] += D[g][1][0];
                    E[g][1] += D[g][1][1];
                }
            }
            // --- x^T += E^T Y^T, tile t -> registers of tile t+1 (the window moves up by 8 rows)
#pragma unroll
            for (int t = NT - 1; t >= 0; --t) {
                const double2 v2 = *reinterpret_cast<const double2 *>(vb + 64 * t);
#pragma unroll
                for (int g = 0; g < NG; ++g) {
                    double m0, m1;
                    dmma884(m0, m1, E[g][0], v2.x, t ? X[g][t][0] : T0[g][0], t ? X[g][t][1] : T0[g][1]);
                    dmma884(X[g][t + 1][0], X[g][t + 1][1], E[g][1], v2.y, m0, m1);
                }
            }
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(bar_empty + 8 * st);
                // the stores of the blocks before this one have long been performed: publishing them
                // here keeps the release fence off the critical path (costs one block of extra lag)
                if (CP && b < btop) prog_publish(mine, (uint32_t)(btop - b));
            }
            // --- tile NT-1 retires (rows 8b + nbw ..), the buffer of tile 0 is refilled
            const int64_t bn = b - (PF2 ? 2 : 1);
            if (fastio && (b << 3) + NBW + 8 <= nrow) {
                double *pr = cb + (b << 3) + 2 * r;
#pragma unroll
                for (int g = 0; g < NG; ++g)
                    *reinterpret_cast<double2 *>(pr + g * ldq8 + NBW) = make_double2(X[g][NT][0], X[g][NT][1]);
                if (bn >= blo) {
                    wait_prev(bn);
                    const double *pl = cb + (bn << 3) + 2 * r;
#pragma unroll
                    for (int g = 0; g < NG; ++g) {
                        const double2 v = CP ? __ldcg(reinterpret_cast<const double2 *>(pl + g * ldq8))
                                             : *reinterpret_cast<const double2 *>(pl + g * ldq8);
                        T0[g][0] = v.x;
                        T0[g][1] = v.y;
                    }
                }
            } else {
#pragma unroll
                for (int g = 0; g < NG; ++g)
                    wy_store2(a, nrow, cb + g * ldq8, 8 * g < ncolrem, (b << 3) + NBW + 2 * r, X[g][NT][0], X[g][NT][1]);
                load_tile0(bn, T0);
            }
            ++it;
        };

        // the window above tile 0: rows 8 btop + 8t ..; beyond the matrix (the whole-matrix launch: every
        // one of them) they read as zero without touching memory, in a sub-range launch they are the rows
        // the rank below handed over
#pragma unroll
        for (int g = 0; g < NG; ++g) {
#pragma unroll
            for (int t = 1; t < NT; ++t) {
                if (RG)
                    wy_load2<CP>(a, nrow, cb + g * ldq8, 8 * g < ncolrem, (btop << 3) + 8 * t + 2 * r, X[g][t][0], X[g][t][1]);
                else
                    X[g][t][0] = X[g][t][1] = 0.0;
            }
            X[g][NT][0] = X[g][NT][1] = 0.0;
            TA[g][0] = TA[g][1] = TB[g][0] = TB[g][1] = 0.0;
        }
        load_tile0(btop, TA);
        if (PF2) {
            load_tile0(btop - 1, TB);
            for (int64_t b = btop; b >= blo; b -= 2) {
                do_block(b, TA);
                if (b - 1 >= blo) do_block(b - 1, TB);
            }
        } else {
            for (int64_t b = btop; b >= blo; --b) do_block(b, TA);
        }
        // --- chain end: tiles 1 .. NT-1 hold rows 8 blo + 8 (t-1) + 2r + {0,1}
#pragma unroll
        for (int g = 0; g < NG; ++g)
#pragma unroll
            for (int t = 1; t < NT; ++t)
                wy_store2(a, nrow, cb + g * ldq8, 8 * g < ncolrem, (blo << 3) + 8 * (t - 1) + 2 * r, X[g][t][0], X[g][t][1]);
        if (CP) {
            __syncwarp();
            if (lane == 0) prog_publish(mine, (uint32_t)(btop - blo + 1));
        }
    }
}

// ---- the kernel ----------------------------------------------------------------------------------------
// grid: CTA c takes slabs [nslab*c/grid, nslab*(c+1)/grid).
//  P = 1: at most NW*NGMAX slabs per CTA; warp w takes n/NW of them, +1 for the first n%NW warps
//         (warps w and w+4 share a sub-partition, so the extras land on different sub-partitions first).
//  P > 1 (few slabs): at most NW/P slabs per CTA; warp w works on slab w/P, chains (w%P) + m P.
// RG: the sub-range build (rows call of SURVEY 8(f) NEXT-3; P = 1 only).  RG = false is the whole-matrix launch.
template <int NBW, int NWARPS, bool RG = false>
__global__ void __launch_bounds__(NWARPS * 32, 1) bt_wy_kernel(const WyArgs a)
{
    using C = WyCfg<NBW, NWARPS>;
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

    // the ring starts as zeros: the skew padding of VA / VB is never written by the copies, and
    // positions of reflectors outside a chain keep finite values (their row and column of T are 0)
    for (int i = threadIdx.x; i < C::OFF_BAR / 8; i += blockDim.x) ring[i] = 0.0;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (threadIdx.x == 0) {
        for (int i = 0; i < NS; ++i) {
            mbar_init(bar_full + 8 * i, 33);           // 32 cp.async arrivals + the bulk copy's expect_tx arrival
            mbar_init(bar_empty + 8 * i, (uint32_t)nact);
        }
        mbar_fence_init();
    }
    __syncthreads();

    if (!RG && a.P > 1) {
        // chain-parallel: `member` = the a.P warps that share slabs; member slots NW / P
        const int grp = warp % a.P, member = warp / a.P, nm = NW / a.P;
        const int base = nmine / nm, extra = nmine % nm;
        const int ng = base + (member < extra ? 1 : 0);
        const int64_t wslab0 = slab0 + (int64_t)member * base + (member < extra ? member : extra);
        if (ng == 0) return;
        if (NGMAX >= 4 && ng == 4)
            wy_consume<C, (NGMAX >= 4 ? 4 : 1), true, false>(a, smem, lane, grp, member, nact, wslab0 << 3, wslab0);
        else if (NGMAX >= 3 && ng == 3)
            wy_consume<C, (NGMAX >= 3 ? 3 : 1), true, false>(a, smem, lane, grp, member, nact, wslab0 << 3, wslab0);
        else if (NGMAX >= 2 && ng == 2)
            wy_consume<C, (NGMAX >= 2 ? 2 : 1), true, false>(a, smem, lane, grp, member, nact, wslab0 << 3, wslab0);
        else
            wy_consume<C, 1, true, false>(a, smem, lane, grp, member, nact, wslab0 << 3, wslab0);
        return;
    }
    if (NWARPS > 8) return;                            // the 16-warp build is chain-parallel only
    const int base = nmine / NW, extra = nmine % NW;
    const int ng = base + (warp < extra ? 1 : 0);
    const int64_t wslab0 = slab0 + (int64_t)warp * base + (warp < extra ? warp : extra);
    if (ng == 0) return;
    const int64_t col0 = wslab0 << 3;
    if (NGMAX >= 4 && ng == 4)
        wy_consume<C, (NGMAX >= 4 ? 4 : 1), false, RG>(a, smem, lane, 0, warp, nact, col0, wslab0);
    else if (NGMAX >= 3 && ng == 3)
        wy_consume<C, (NGMAX >= 3 ? 3 : 1), false, RG>(a, smem, lane, 0, warp, nact, col0, wslab0);
    else if (NGMAX >= 2 && ng == 2)
        wy_consume<C, (NGMAX >= 2 ? 2 : 1), false, RG>(a, smem, lane, 0, warp, nact, col0, wslab0);
    else if (NWARPS <= 8)
        wy_consume<C, 1, false, RG>(a, smem, lane, 0, warp, nact, col0, wslab0);
}

// ---- host side -----------------------------------------------------------------------------------------
// warps per slab: with fewer slabs than warp slots, P warps share a slab on different chains
inline int wy_pick_P(int64_t nslab, int64_t K0, int nsm, int nw, int maxP)
{
    const int64_t grid = nslab < nsm ? nslab : nsm;
    const int64_t spc = (nslab + grid - 1) / grid;     // most slabs per CTA when the grid is one wave
    int P = 1;
    while (2 * P <= maxP && spc * 2 * P <= nw && 4 * P <= K0) P *= 2;
    return nslab <= (int64_t)nsm * nw ? P : 1;
}

// Busiest sub-partition of a CTA that holds n slabs with P warps per slab group, in slab-passes: the 8
// warps form 8/P groups, group m = warps mP .. mP+P-1 takes n/(8/P) slabs (+1 for the first ones) and each
// of its warps walks 1/P of their chains; warp w issues on sub-partition w % 4, whose DMMA pipe is the
// resource the kernel is bound by.
inline double wy_smsp_load(int P, int64_t n)
{
    const int nm = 8 / P;
    double load[4] = {0, 0, 0, 0};
    for (int w = 0; w < 8; ++w) {
        const int m = w / P;
        load[w & 3] += (double)(n / nm + (m < n % nm ? 1 : 0)) / P;
    }
    double mx = 0;
    for (int s = 0; s < 4; ++s) mx = load[s] > mx ? load[s] : mx;
    return mx;
}
// Real kernel, one wave: P in {1, 2, 4} for partial spectra (5-16 slabs per SM).  Measured on B200
// (N = 8192, nbw 64, n slabs per SM; TFLOP/s for P = 1 / 2 / 4):
//   n = 5: 15.3 / 19.8 / 25.9    6: 18.8 / 23.7 / 26.9    7: 22.3 / 23.6 / 27.1
//   n = 9: 21.0 / 25.7    10: 23.2 / 28.4    11: 25.5 / 27.9    12: 27.8 / 29.8    13: 24.2 / 26.7    14: 26.0 / 28.7
//   n = 15: 27.8 / 27.5   16: 29.6 / 29.4
// Two things are at work: the balance of the four sub-partitions (wy_smsp_load) and the number of slabs a
// warp holds -- warps with 3-4 slabs run the DMMA pipe better than warps with 1-2, and P warps that share a
// group of slabs hold P times as many each.  Hence: up to 8 slabs P = 4, 9-14 slabs P = 2, above that P = 1.
inline int wy_pick_P_real(int64_t nslab, int64_t K0, int nsm, int ngmax, int maxP)
{
    const int64_t grid = nslab < nsm ? nslab : nsm;
    const int64_t n = (nslab + grid - 1) / grid;
    if (n > 8 * (int64_t)ngmax) return 1;              // more than one wave of the P = 1 launch
    auto ok = [&](int P) { return P <= maxP && 4 * P <= K0 && n <= (int64_t)(8 / P) * ngmax; };
    if (n <= 8) return ok(4) ? 4 : ok(2) ? 2 : 1;
    if (n <= 14) return ok(2) ? 2 : 1;
    return (ok(2) && wy_smsp_load(2, n) * 1.03 < wy_smsp_load(1, n)) ? 2 : 1;
}

// Complex kernel (P <= 2): up to 4 slabs per SM the rule of round 1 (one slab per warp, two warps per slab:
// 18.7 -> 25.4 TFLOP/s on config 3); above that, while the P = 2 launch still fits in one wave
// (n <= 4 ngmax), P = 2 when it lowers the busiest sub-partition.
inline int wy_pick_P_cplx(int64_t nslab, int64_t K0, int nsm, int ngmax, int maxP)
{
    const int base = wy_pick_P(nslab, K0, nsm, 8, maxP);
    if (base > 1) return base;
    const int64_t grid = nslab < nsm ? nslab : nsm;
    const int64_t n = (nslab + grid - 1) / grid;
    if (maxP >= 2 && 8 <= K0 && n > 4 && n <= 4 * (int64_t)ngmax && wy_smsp_load(2, n) * 1.03 < wy_smsp_load(1, n)) return 2;
    return 1;
}

// launch plan of the main kernel (pure host arithmetic; exported as elpa2_bt_plan for the CPU tests)
struct WyPlan {
    int64_t grid;        // CTAs
    int nwarps;          // warps per CTA: 8, or 16 (real, few columns)
    int P;               // warps per slab group (chains per pass)
    int64_t nslab;       // slabs of 8 columns
    int64_t per_cta;     // most slabs a CTA can take
};
inline WyPlan wy_plan(bool cplx, int nbw, int64_t N, int64_t nev, int nsm, int force_P, int force_nw)
{
    const int64_t K0 = wy_nchains(N, nbw);
    WyPlan pl;
    pl.nslab = (nev + 7) >> 3;
    const int ngmax8 = cplx ? (nbw <= 64 ? 2 : 1) : (nbw <= 64 ? 4 : nbw <= 128 ? 2 : 1);
    const bool many_warps = !cplx && nbw <= 64 && force_P == 0 && force_nw != 8 && pl.nslab <= (int64_t)nsm * 4 && K0 >= 16;
    pl.nwarps = many_warps ? 16 : 8;
    // a chain-parallel group needs at least two ring stages of its own: P <= NS / 2
    const int ns = cplx ? (nbw <= 64 ? 8 : 4) : ((8 * 16 * (nbw + 8) * 8 <= 216 * 1024) ? 8 : 4);
    const int maxP = cplx ? 2 : (ns >= 8 ? 4 : 2);
    if (force_P > maxP) force_P = maxP;
    pl.P = many_warps ? 4
           : force_P > 0 ? force_P
           : cplx ? wy_pick_P_cplx(pl.nslab, K0, nsm, ngmax8, maxP)
                  : wy_pick_P_real(pl.nslab, K0, nsm, ngmax8, maxP);
    // (the 16-warp build walks one slab per warp)
    pl.per_cta = (int64_t)(pl.nwarps / pl.P) * (many_warps ? 1 : ngmax8);
    const int64_t waves = (pl.nslab + nsm * pl.per_cta - 1) / (nsm * pl.per_cta);
    pl.grid = nsm * waves;                            // a multiple of the SM count ...
    if (pl.grid > pl.nslab) pl.grid = pl.nslab;       // ... unless there are fewer slabs than that
    return pl;
}

// bytes of scratch the two kernels share: -T factors, then the chain-progress counters
template <int NBW>
size_t wy_tn_bytes(int64_t N)
{
    return (size_t)wy_nblocks(N, NBW) * WyCfg<NBW>::YBLK * sizeof(double);
}
template <int NBW>
size_t wy_scratch_bytes(int64_t N, int64_t nev)
{
    const size_t prog = (size_t)((nev + 7) >> 3) * (size_t)wy_nchains(N, NBW) * sizeof(uint32_t);
    return wy_tn_bytes<NBW>(N) + ((prog + 255) & ~(size_t)255);
}

template <int NBW, int NWARPS, bool RG = false>
cudaError_t launch_wy_main(const WyArgs &a, const WyPlan &pl, cudaStream_t st)
{
    using C = WyCfg<NBW, NWARPS>;
    auto kern = bt_wy_kernel<NBW, NWARPS, RG>;
    {
        cudaError_t e = set_max_smem((const void *)kern, C::SMEM_BYTES);
        if (e != cudaSuccess) return e;
    }
    kern<<<(unsigned)pl.grid, NWARPS * 32, C::SMEM_BYTES, st>>>(a);
    return cudaGetLastError();
}

// Sub-range of a launch: the chains [kb, ke) restricted to the blocks whose first row
// lies in the rows [row0, row0 + nown) this caller owns; its q holds the rows [row0, row_end).  row0 a
// multiple of 8.  The whole matrix: kb = 0, ke = -1 (= K0), row0 = 0, nown = row_end = N.
struct WyRange {
    int64_t kb = 0, ke = -1, row0 = 0, nown = -1, row_end = -1;
    bool whole() const { return ke < 0; }
};
// chains of the range that have a block here, block bounds (host arithmetic shared by real and complex)
inline void wy_range_resolve(const WyRange &r, int64_t N, int nbw, int64_t &kb, int64_t &ke, int64_t &b_top, int64_t &b_bot,
                             int64_t &row_end)
{
    const int64_t K0 = wy_nchains(N, nbw), bhi = wy_bhi(N);
    if (r.whole()) {
        kb = 0, ke = K0, b_top = bhi, b_bot = 0, row_end = N;
        return;
    }
    b_bot = r.row0 >> 3;
    b_top = ((r.row0 + r.nown) >> 3) - 1;
    if (r.row0 + r.nown >= N || b_top > bhi) b_top = bhi;
    row_end = r.row_end;
    kb = r.kb;
    ke = r.ke < K0 ? r.ke : K0;
    const int64_t klast = b_top / (nbw >> 3);          // chains beyond it start below this range
    if (ke > klast + 1) ke = klast + 1;
    if (ke < kb) ke = kb;
}
template <int NBW>
size_t wy_tn_bytes_range(int64_t N, int64_t kb, int64_t ke)
{
    return (size_t)(wy_base(N, NBW, ke) - wy_base(N, NBW, kb)) * WyCfg<NBW>::YBLK * sizeof(double);
}

// force_P > 0 overrides the number of warps per slab of the 8-warp kernel; force_nw = 8 keeps the
// 16-warp kernel (few columns: 4 warps per slab, 128 registers each) from being chosen.
// A sub-range launch (rg) runs P = 1 on the 8-warp kernel; `scratch` then holds the chains [kb, ke) only.
template <int NBW>
cudaError_t launch_wy(int64_t N, int64_t nev, const double *hh_v, const double *hh_tau, double *q, int64_t ldq,
                      int align16, int nsm, void *scratch, cudaStream_t st, int force_P = 0, int force_nw = 0,
                      const WyRange &rg = WyRange())
{
    using C = WyCfg<NBW>;
    const int64_t K0 = wy_nchains(N, C::NBW);
    const int64_t nslab = (nev + 7) >> 3;
    WyArgs a;
    wy_range_resolve(rg, N, NBW, a.kb, a.ke, a.b_top, a.b_bot, a.row_end);
    if (a.ke <= a.kb) return cudaSuccess;
    if (!rg.whole()) force_P = 1, force_nw = 8;
    const size_t tn_bytes = rg.whole() ? wy_tn_bytes<NBW>(N) : wy_tn_bytes_range<NBW>(N, a.kb, a.ke);
    double *tn = (double *)scratch - wy_base(N, NBW, a.kb) * C::YBLK;      // addressed by global block ids
    uint32_t *prog = (uint32_t *)((char *)scratch + tn_bytes);
    const WyPlan pl = wy_plan(false, NBW, N, nev, nsm, force_P, force_nw);
    const int P = pl.P;
    cudaError_t e;
    if (P > 1) {
        e = cudaMemsetAsync(prog, 0, (size_t)nslab * K0 * sizeof(uint32_t), st);
        if (e != cudaSuccess) return e;
    }
    const dim3 pgrid((unsigned)((wy_bhi(N) + C::PW) / C::PW), (unsigned)(a.ke - a.kb));
    wy_prepass_kernel<NBW><<<pgrid, C::PW * 32, 0, st>>>(N, hh_v, hh_tau, tn, a.kb);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    a.N = N;
    a.nev = nev;
    a.ldq = ldq;
    a.hh_v = hh_v;
    a.hh_tau = hh_tau;
    a.q = q - rg.row0;                                  // addressed by global row indices
    a.tn = tn;
    a.prog = prog;
    a.align16 = align16;
    a.P = P;
    if (!rg.whole()) return launch_wy_main<NBW, 8, true>(a, pl, st);
    if (pl.nwarps == 16) return launch_wy_main<(NBW <= 64 ? NBW : 64), 16>(a, pl, st);
    return launch_wy_main<NBW, 8>(a, pl, st);
}

}  // namespace elpa2bt
