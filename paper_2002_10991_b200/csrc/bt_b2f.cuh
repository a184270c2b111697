// bt_b2f.cuh -- SURVEY.md 8(f) NEXT-2: band -> full back-transformation of the eigenvectors (Eq. 6e,
// C = P* Y) on the FP64 tensor cores (DMMA m8n8k4), real FP64, sm_100a.
// What it computes: include/elpa2_bt.h, reading R15 of DESIGN.md:
//      q <- H_0 H_1 ... H_{Nv-1} q,   H_j = I - tau_j v_j v_j^T on rows j+nbw .. N-1,  Nv = N - nbw - 1.
// The paper names this step a BLAS-3 (cuBLAS) step and, with 6a, "the first target for further ...
// optimization".  Here it is ONE hand-written GEMM-class kernel, not a sequence of
// library GEMMs:
//
//  * Blocks of NB = 64 consecutive reflectors, Q_p = H_{64p} .. H_{64p+63} = I - V_p T_p V_p^T (compact
//    WY, T_p upper triangular: T[i][i] = tau_i, T[:i, i] = -tau_i T[:i,:i] (V[:, :i]^T v_i); the prepass
//    kernel b2f_tfactor_kernel writes -T_p).  q <- Q_0 (Q_1 ( .. Q_{npb-1} q)): block npb-1 first.
//  * Applying Q_p is  W = V_p^T q  (64 x cols, K = rows),  U = (-T_p) W,  q += V_p U  (K = 64).  The two
//    big products of CONSECUTIVE blocks are fused into one pass over q ("look-ahead"): pass P reads a
//    16-row group of q once, updates it with block P (q += V_P U_P), feeds the updated rows straight
//    into the dot product of block P-1 (W_{P-1} += V_{P-1}^T q) and writes it once.  q traffic per
//    block is one read + one write instead of two reads + one write: 2*8 bytes per 4*64 flops and
//    column, AI = 16 flop/B, above the ridge (5.7).
//  * Everything is computed transposed so that "column of q" sits on the M index of every fragment and
//    the C fragment of one product is, register for register, the A fragment of the next (the zero-
//    shuffle fragment chaining of bt_wy.cuh): W^T = q^T V, U^T = W^T (-T)^T, q^T += U^T V^T.
//    Lane (gq, r) = (lane / 4, lane % 4) holds rows 4r .. 4r+3 of column gq of a 16-row group (32
//    contiguous bytes; the four lanes of a column cover one 128-byte line).
//  * V tiles (16 rows x 64 reflectors of block P and of block P-1) are staged by the warps in turn
//    with 16-byte cp.async (zero fill beyond N / Nv) into a 4-stage shared-memory ring
//    [reflector][18 doubles]: the row stride 18 makes both B-fragment access patterns (LDS.128)
//    bank-conflict free.  Completion on mbarriers, no CTA barrier in the loop.
//  * A warp owns 1 or 2 slabs of 8 columns for ALL passes: W and U (2 x 16 doubles per slab) live in
//    registers.  Its rows of q arrive through a private 6-stage shared-memory ring filled by its own
//    cp.async copies four items ahead (no register is tied up by a load in flight, and no scoreboard is
//    shared between the q stream and the B-fragment loads); updated rows go back to global memory
//    straight from the C fragments.  CTAs never communicate; a CTA walks its slabs in rounds of up to 16.
// Wasted tensor work: only the zero upper triangle of the first 64 rows of each block (0.2 % at
// N = 32768) and the 64 x 64 T product per pass.
#pragma once
#include "bt_common.cuh"
#include "bt_wy.cuh"        // dmma884, cp_async_mbar_arrive_noinc_wy

namespace elpa2bt {

struct B2fCfg {
    static constexpr int NB = 64;                     // reflectors per block
    static constexpr int GR = 16;                     // rows per group (one ring stage)
    static constexpr int S = 18;                      // smem row stride per reflector (doubles): S/2 odd
    static constexpr int PANEL = NB * S;              // doubles per panel tile
    static constexpr int STAGE_DOUBLES = 2 * PANEL;   // panel 0: block P (update), panel 1: block P-1 (dot)
    static constexpr int NS = 4, LGNS = 2, LAG = 2;   // V ring (shared by the CTA); 8 stages / 4 ahead measured the same
    static constexpr int NW = 8;                      // warps per CTA
    static constexpr int NGMAX = 2;                   // slabs per warp
    static constexpr int QS = 18;                     // q tile: [column][QS doubles], QS/2 odd
    static constexpr int QTILE = 8 * NGMAX * QS;      // doubles per q tile (one warp, one item)
    static constexpr int NSQ = 6, DQ = 4;             // q ring per warp: stages, items fetched ahead (DQ <= 4, see b2f_consume)
    static constexpr int OFF_Q = NS * STAGE_DOUBLES * 8;
    static constexpr int OFF_BAR = OFF_Q + NW * NSQ * QTILE * 8;
    static constexpr int SMEM_BYTES = OFF_BAR + 2 * NS * 8;
    static_assert(SMEM_BYTES <= 227 * 1024, "shared memory");
};

// N, ldq and ldv count DOUBLES per column (= elements x ew): the complex kernel (bt_b2fz.cuh) sees its
// interleaved N x Nv matrix as a real 2N x Nv one, so staging, the q ring and the tile stores are shared.
struct B2fArgs {
    int64_t N, nev, ldq, ldv, Nv;
    int nbw;               // in elements
    int ew;                // doubles per element: 1 real, 2 complex
    const double *hv;      // N x Nv column-major, ldv
    const double *tneg;    // npb x 64 x 64 elements, row-major: tneg[p][i][k] = -T_p[i][k]
    double *q;
    int align16;           // q base and ldq*8 are 16-byte aligned (always 1 for complex)
};

__host__ __device__ __forceinline__ int64_t b2f_nblocks(int64_t Nv) { return (Nv + B2fCfg::NB - 1) / B2fCfg::NB; }

// ---- prepass: -T_p of every block (plain FP64; 0.1 % of the work of a call) -----------------------------
// One CTA (256 threads) per block p.  S = V^T V over rows i0 .. N-1 (thread (ty, tx) owns the 4 x 4
// sub-block S[4ty.., 4tx..]; V staged 16 rows at a time), then the larft recurrence column by column.
__global__ void __launch_bounds__(256) b2f_tfactor_kernel(int64_t N, int64_t Nv, int nbw, const double *__restrict__ hv,
                                                          int64_t ldv, const double *__restrict__ tau,
                                                          double *__restrict__ tneg)
{
    constexpr int NB = B2fCfg::NB, RC = 16, SV = NB + 1;
    __shared__ double Vs[RC * SV];                    // Vs[row][refl]
    __shared__ double Sm[NB * SV];                    // Gram matrix, then T
    __shared__ double taus[NB];
    const int tid = threadIdx.x;
    const int64_t p = blockIdx.x;
    const int64_t j0 = p * NB;
    const int nb = (int)((Nv - j0 < NB) ? Nv - j0 : NB);
    const int64_t i0 = j0 + nbw;
    const int ty = tid >> 4, tx = tid & 15;
    double acc[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b] = 0.0;
    if (tid < NB) taus[tid] = (tid < nb) ? tau[j0 + tid] : 0.0;
    for (int64_t rb = i0; rb < N; rb += RC) {
        // rows rb .. rb+15, lanes along rows (contiguous in hv)
        for (int idx = tid; idx < RC * NB; idx += 256) {
            const int c = idx >> 4, rr = idx & 15;
            const int64_t row = rb + rr;
            Vs[rr * SV + c] = (c < nb && row < N) ? hv[row + (j0 + c) * ldv] : 0.0;
        }
        __syncthreads();
#pragma unroll 4
        for (int rr = 0; rr < RC; ++rr) {
            double a4[4], b4[4];
#pragma unroll
            for (int a = 0; a < 4; ++a) a4[a] = Vs[rr * SV + 4 * ty + a];
#pragma unroll
            for (int b = 0; b < 4; ++b) b4[b] = Vs[rr * SV + 4 * tx + b];
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) acc[a][b] = fma(a4[a], b4[b], acc[a][b]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) Sm[(4 * ty + a) * SV + 4 * tx + b] = acc[a][b];
    __syncthreads();
    // larft (forward, columnwise), in place: column i of T overwrites column i of S above the diagonal;
    // thread r < i owns T[r][i] = -tau_i sum_{k = r}^{i-1} T[r][k] S[k][i]  (T[r][k], k < i, already final)
    __shared__ double colS[NB];
    for (int i = 0; i < NB; ++i) {
        if (tid < i) colS[tid] = Sm[tid * SV + i];
        __syncthreads();
        if (tid < i) {
            double s = 0.0;
            for (int k = tid; k < i; ++k) s = fma((k == tid) ? taus[tid] : Sm[tid * SV + k], colS[k], s);
            Sm[tid * SV + i] = -taus[i] * s;
        }
        __syncthreads();
    }
    // -T, row-major 64 x 64, zeros below the diagonal
    double *out = tneg + p * (NB * NB);
    for (int idx = tid; idx < NB * NB; idx += 256) {
        const int i = idx >> 6, k = idx & 63;
        out[idx] = (k > i) ? -Sm[i * SV + k] : (k == i ? -taus[i] : 0.0);
    }
}

// ---- the sequence of ring items: pass P = npb .. 0, groups g = g_lo(P) .. g_hi ---------------------------
// pass P updates with block P (P < npb; rows >= i0(P)) and accumulates the dot product of block P-1
// (P >= 1; rows >= i0(P-1) = i0(P) - 64).  i0(p) = 64 p + nbw is a multiple of 16.
struct B2fCursor {
    int64_t P, g;
};
__device__ __forceinline__ int64_t b2f_glo(int64_t P, int nbw, int ew = 1)
{
    const int64_t pb = P >= 1 ? P - 1 : 0;
    return ((pb * B2fCfg::NB + nbw) * ew) >> 4;
}

// stage one item (whole warp): panel 0 = V_P rows of group g (if the group is inside block P),
// panel 1 = V_{P-1}.  1024 chunks of 16 bytes; lanes run along the 8 chunks of a reflector's 128 bytes,
// four reflectors per instruction.  Warp-uniform fast path (group inside the matrix, block full): one
// cp.async and one pointer increment per chunk.
__device__ __forceinline__ void b2f_stage(const B2fArgs &a, double *stage, uint32_t bar_full, int64_t P, int64_t g,
                                          int64_t npb, int lane)
{
    constexpr int NB = B2fCfg::NB, S = B2fCfg::S;
    const int64_t row0 = g << 4;
    const int ch = lane & 7, lr = lane >> 3;
    const int64_t row = row0 + 2 * ch;
    const bool rows_full = row0 + 16 <= a.N;          // warp-uniform
    const int64_t ld4 = a.ldv << 2;
#pragma unroll
    for (int panel = 0; panel < 2; ++panel) {
        const int64_t blk = P - panel;
        const bool on = (panel == 0) ? (P < npb && row0 >= (P * NB + a.nbw) * a.ew) : (P >= 1);
        if (!on) continue;                            // warp-uniform
        const double *src = a.hv + row + (blk * NB + lr) * a.ldv;
        const uint32_t dst = smem_u32(stage + panel * B2fCfg::PANEL + lr * S + 2 * ch);
        if (rows_full && (blk + 1) * NB <= a.Nv) {
#pragma unroll
            for (int t = 0; t < NB / 4; ++t) {
                cp_async16(dst + t * (4 * S * 8), src, 16u);
                src += ld4;
            }
        } else {
            const uint32_t nbytes = (row + 1 < a.N) ? 16u : (row < a.N ? 8u : 0u);
#pragma unroll 4
            for (int t = 0; t < NB / 4; ++t) {
                const bool ok = (blk * NB + 4 * t + lr < a.Nv) && nbytes;
                cp_async16(dst + t * (4 * S * 8), ok ? src : a.hv, ok ? nbytes : 0u);
                src += ld4;
            }
        }
    }
    cp_async_mbar_arrive_noinc_wy(bar_full);
}

// q rows 16 g + 4 r .. + 3 of this lane's column go back to global memory from the C fragments
__device__ __forceinline__ void b2f_store4(const B2fArgs &a, double *colp, bool colok, int64_t row, bool fast,
                                           const double (&y)[4])
{
    if (fast) {
        *reinterpret_cast<double2 *>(colp + row) = make_double2(y[0], y[1]);
        *reinterpret_cast<double2 *>(colp + row + 2) = make_double2(y[2], y[3]);
        return;
    }
#pragma unroll
    for (int e = 0; e < 4; ++e)
        if (colok && row + e < a.N) colp[row + e] = y[e];
}

// One warp's 16-row tile of q (8 NG columns) into its private shared-memory tile [column][QS doubles]:
// BYTES = 16 (q base and ldq*8 16-byte aligned) or 8.  Lanes run along the 128 bytes of a column; zero fill
// beyond N and beyond nev.
template <int NG, int BYTES>
__device__ __forceinline__ void b2f_fetch_q(const B2fArgs &a, double *tile, int64_t col0, int64_t g, int lane)
{
    constexpr int QS = B2fCfg::QS;
    constexpr int CPC = 128 / BYTES;                  // chunks per column
    constexpr int CPI = 32 / CPC;                     // columns per instruction
    const int ch = lane % CPC, cq = lane / CPC;
    const int64_t row = (g << 4) + ch * (BYTES / 8);
    const bool rows_full = (g << 4) + 16 <= a.N;
    const bool cols_full = col0 + 8 * NG <= a.nev;
    const double *src = a.q + (col0 + cq) * a.ldq + row;
    const uint32_t dst = smem_u32(tile + cq * QS + ch * (BYTES / 8));
    const int64_t ldc = a.ldq * CPI;
    if (rows_full && cols_full) {
#pragma unroll
        for (int t = 0; t < 8 * NG / CPI; ++t) {
            if (BYTES == 16)
                cp_async16(dst + t * (CPI * QS * 8), src, 16u);
            else
                cp_async8(dst + t * (CPI * QS * 8), src, 8u);
            src += ldc;
        }
    } else {
        uint32_t nbytes = 0;
        if (BYTES == 16)
            nbytes = (row + 1 < a.N) ? 16u : (row < a.N ? 8u : 0u);
        else
            nbytes = (row < a.N) ? 8u : 0u;
#pragma unroll
        for (int t = 0; t < 8 * NG / CPI; ++t) {
            const bool ok = (col0 + cq + t * CPI < a.nev) && nbytes;
            if (BYTES == 16)
                cp_async16(dst + t * (CPI * QS * 8), ok ? src : a.q, ok ? nbytes : 0u);
            else
                cp_async8(dst + t * (CPI * QS * 8), ok ? src : a.q, ok ? nbytes : 0u);
            src += ldc;
        }
    }
}

// ---- a warp with NG slabs of 8 columns, all passes ---------------------------------------------------------
template <int NG>
__device__ __forceinline__ void b2f_consume(const B2fArgs &a, unsigned char *smem, const int lane, const int warp,
                                            const int member, const int nmem, const int64_t col0)
{
    using C = B2fCfg;
    constexpr int NB = C::NB, S = C::S, NSP = C::NS, LAG = C::LAG, QS = C::QS, NSQ = C::NSQ, DQ = C::DQ;
    double *ring = reinterpret_cast<double *>(smem);
    double *qring = reinterpret_cast<double *>(smem + C::OFF_Q) + (size_t)warp * NSQ * C::QTILE;
    const uint32_t bar_full = smem_u32(smem + C::OFF_BAR);
    const uint32_t bar_empty = bar_full + C::NS * 8;
    const int gq = lane >> 2, r = lane & 3;
    const int64_t N = a.N;
    const int64_t npb = b2f_nblocks(a.Nv);
    const int64_t ghi = (N - 1) >> 4;

    double *const cb = a.q + (col0 + gq < a.nev ? col0 + gq : 0) * a.ldq;
    const int64_t ldq8 = a.ldq << 3;
    const int64_t ncolrem = a.nev - col0 - gq;          // column g is valid iff 8g < ncolrem
    const bool allcols = a.align16 && (col0 + 8 * NG <= a.nev);

    // two cursors into the item sequence, kept identically by every warp of the CTA: pc = the V tile the
    // warp on duty stages now (item it + NSP - LAG), qc = the q tile this warp fetches now (item it + DQ)
    B2fCursor pc = {npb, b2f_glo(npb, a.nbw)}, qc = pc;
    auto advance = [&](B2fCursor &c) {
        if (c.P < 0) return;
        if (c.g < ghi) {
            ++c.g;
        } else {
            --c.P;
            c.g = b2f_glo(c.P, a.nbw);
        }
    };
    auto fetch_q = [&](int qst) {
        if (qc.P >= 0) {
            if (a.align16)
                b2f_fetch_q<NG, 16>(a, qring + qst * C::QTILE, col0, qc.g, lane);
            else
                b2f_fetch_q<NG, 8>(a, qring + qst * C::QTILE, col0, qc.g, lane);
        }
        cp_async_commit();                              // one group per item, empty past the end
        advance(qc);
    };
    uint32_t it = 0;
    int duty = 0, qst_in = 0, qst_out = 0;              // q ring positions of item it + DQ / item it
    // prologue: V tiles of items 0 .. NSP-LAG-1 into fresh stages, q tiles of items 0 .. DQ-1
    for (int i = 0; i < NSP - LAG; ++i) {
        if (duty == member && pc.P >= 0)
            b2f_stage(a, ring + i * C::STAGE_DOUBLES, bar_full + 8 * i, pc.P, pc.g, npb, lane);
        advance(pc);
        duty = (duty + 1 == nmem) ? 0 : duty + 1;
    }
    for (int i = 0; i < DQ; ++i) {
        fetch_q(qst_in);
        qst_in = (qst_in + 1 == NSQ) ? 0 : qst_in + 1;
    }

    double W[NG][8][2], U[NG][8][2];
#pragma unroll
    for (int s = 0; s < NG; ++s)
#pragma unroll
        for (int i = 0; i < 8; ++i) W[s][i][0] = W[s][i][1] = U[s][i][0] = U[s][i][1] = 0.0;

    int64_t P = npb, g = b2f_glo(npb, a.nbw);
    while (P >= 0) {
        // --- staging duty for the V ring (rotates over the warps of the CTA, bt_wy.cuh)
        {
            const uint32_t seq = it + NSP - LAG;
            if (duty == member && pc.P >= 0) {
                const uint32_t st = seq & (NSP - 1);
                if (seq >= (uint32_t)NSP) mbar_wait(bar_empty + 8 * st, ((seq - NSP) >> C::LGNS) & 1);
                b2f_stage(a, ring + st * C::STAGE_DOUBLES, bar_full + 8 * st, pc.P, pc.g, npb, lane);
            }
            advance(pc);
            duty = (duty + 1 == nmem) ? 0 : duty + 1;
        }
        // --- this warp's q tile of item it + DQ (its stage was read DQ - NSQ items ago; the __syncwarp at the
        //     end of every item orders those reads before these copies).  Rows an earlier pass wrote were
        //     written by lanes of this warp at least one __syncwarp ago, and a tile fetched ahead across a
        //     pass boundary holds one of the first DQ <= 4 groups of the next pass: rows above block P, which
        //     the pass in flight does not write.
        fetch_q(qst_in);
        qst_in = (qst_in + 1 == NSQ) ? 0 : qst_in + 1;
        asm volatile("cp.async.wait_group %0;" ::"n"(DQ) : "memory");      // the tile of item `it` has landed (own copies)
        __syncwarp();                                                     // ... and every other lane's
        const uint32_t st = it & (NSP - 1), ph = (it >> C::LGNS) & 1;
        mbar_wait(bar_full + 8 * st, ph);
        const double *pa = ring + st * C::STAGE_DOUBLES;      // V_P tile
        const double *pb = pa + C::PANEL;                     // V_{P-1} tile
        const bool has_upd = (P < npb) && ((g << 4) >= P * NB + a.nbw);   // warp-uniform
        const bool has_dot = P >= 1;

        // --- rows 4r .. 4r+3 of column gq of every slab: n-tile 0 = rows 2n (C fragment Y0 = rows 4r, 4r+2),
        //     n-tile 1 = rows 2n+1 (Y1 = rows 4r+1, 4r+3)
        double Y0[NG][2], Y1[NG][2];
        {
            const double *qt = qring + qst_out * C::QTILE + gq * QS + 4 * r;
#pragma unroll
            for (int s = 0; s < NG; ++s) {
                const double2 u = *reinterpret_cast<const double2 *>(qt + 8 * s * QS);
                const double2 w = *reinterpret_cast<const double2 *>(qt + 8 * s * QS + 2);
                Y0[s][0] = u.x, Y1[s][0] = u.y, Y0[s][1] = w.x, Y1[s][1] = w.y;
            }
        }
        qst_out = (qst_out + 1 == NSQ) ? 0 : qst_out + 1;

        if (has_upd) {
            // --- q^T += U^T V_P^T: K = 64 reflectors, chunk (i, e): k-slot r = reflector 8i + 2r + e
            const double *bp = pa + (2 * r) * S + 2 * gq;
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const double2 b = *reinterpret_cast<const double2 *>(bp + (8 * i + e) * S);
#pragma unroll
                    for (int s = 0; s < NG; ++s) {
                        dmma884(Y0[s][0], Y0[s][1], U[s][i][e], b.x, Y0[s][0], Y0[s][1]);
                        dmma884(Y1[s][0], Y1[s][1], U[s][i][e], b.y, Y1[s][0], Y1[s][1]);
                    }
                }
        }
        if (has_dot) {
            // --- W^T += q^T V_{P-1}: K = 16 rows, chunk e: k-slot r = row 4r + e; n-tile i = reflectors 8i + n.
            //     Two n-tiles at a time: 2 NG independent accumulators in rotation (splitting further -- four
            //     chains for a one-slab warp -- was measured and changed nothing)
            const double *bp = pb + gq * S + 4 * r;
#pragma unroll
            for (int i = 0; i < 8; i += 2) {
                const double2 b00 = *reinterpret_cast<const double2 *>(bp + 8 * i * S);
                const double2 b01 = *reinterpret_cast<const double2 *>(bp + 8 * i * S + 2);
                const double2 b10 = *reinterpret_cast<const double2 *>(bp + 8 * (i + 1) * S);
                const double2 b11 = *reinterpret_cast<const double2 *>(bp + 8 * (i + 1) * S + 2);
                const double bv[2][4] = {{b00.x, b00.y, b01.x, b01.y}, {b10.x, b10.y, b11.x, b11.y}};
#pragma unroll
                for (int e = 0; e < 4; ++e)
#pragma unroll
                    for (int d = 0; d < 2; ++d)
#pragma unroll
                        for (int s = 0; s < NG; ++s) {
                            const double ya = (e == 0) ? Y0[s][0] : (e == 1) ? Y1[s][0] : (e == 2) ? Y0[s][1] : Y1[s][1];
                            dmma884(W[s][i + d][0], W[s][i + d][1], ya, bv[d][e], W[s][i + d][0], W[s][i + d][1]);
                        }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * st);
        if (has_upd) {
            const int64_t row = (g << 4) + 4 * r;
            const bool fast = allcols && ((g << 4) + 16 <= N);    // warp-uniform
#pragma unroll
            for (int s = 0; s < NG; ++s) {
                const double y[4] = {Y0[s][0], Y1[s][0], Y0[s][1], Y1[s][1]};
                b2f_store4(a, cb + s * ldq8, 8 * s < ncolrem, row, fast, y);
            }
        }
        ++it;
        if (has_dot && g == ghi) {
            // --- end of pass: U^T = W^T (-T_{P-1})^T.  n-tile i' = reflectors 8i' + n, k chunk (i, e): k-slot r =
            //     reflector 8i + 2r + e; B[k][n] = -T[8i' + n][k], zero for k-tiles i < i' (T upper triangular)
            const double *tp = a.tneg + (P - 1) * (NB * NB) + gq * NB + 2 * r;
#pragma unroll
            for (int ip = 0; ip < 8; ++ip) {
                double c0[NG], c1[NG];
#pragma unroll
                for (int s = 0; s < NG; ++s) c0[s] = c1[s] = 0.0;
#pragma unroll
                for (int i = ip; i < 8; ++i) {
                    const double2 b = __ldg(reinterpret_cast<const double2 *>(tp + 8 * ip * NB + 8 * i));
#pragma unroll
                    for (int s = 0; s < NG; ++s) {
                        dmma884(c0[s], c1[s], W[s][i][0], b.x, c0[s], c1[s]);
                        dmma884(c0[s], c1[s], W[s][i][1], b.y, c0[s], c1[s]);
                    }
                }
#pragma unroll
                for (int s = 0; s < NG; ++s) {
                    U[s][ip][0] = c0[s];
                    U[s][ip][1] = c1[s];
                }
            }
#pragma unroll
            for (int s = 0; s < NG; ++s)
#pragma unroll
                for (int i = 0; i < 8; ++i) W[s][i][0] = W[s][i][1] = 0.0;
        }
        if (g < ghi) {
            ++g;
        } else {
            --P;
            g = b2f_glo(P, a.nbw);
        }
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
}

// slabs of the next round: rem slabs and `units` slab-passes (of 4 slabs) are left for `left` rounds
__device__ __forceinline__ int64_t b2f_round(int64_t rem, int64_t left, int64_t &units)
{
    const int64_t c = (units + left - 1) / left;       // this round's share of the slab-passes
    const int64_t later = 4 * (units - c);             // what the later rounds can take
    int64_t nr = (rem + left - 1) / left;
    if (nr < rem - later) nr = rem - later;
    if (nr > 4 * c) nr = 4 * c;
    if (nr > rem) nr = rem;
    units -= c;
    return nr;
}

// ---- the kernel ----------------------------------------------------------------------------------------------
// grid: CTA c takes slabs [nslab*c/grid, nslab*(c+1)/grid) and walks them in rounds of up to NW*NGMAX = 16;
// (equal-sized rounds); in a round warp w takes n/8 slabs, +1 for the first n%8 warps (warps w and w+4 share a sub-partition).
// A round is one full sequence of passes; the V ring is drained and re-initialised between rounds.
__global__ void __launch_bounds__(256, 1) bt_b2f_kernel(const B2fArgs a)
{
    using C = B2fCfg;
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t bar_full = smem_u32(smem + C::OFF_BAR);
    const uint32_t bar_empty = bar_full + C::NS * 8;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t nslab = (a.nev + 7) >> 3;
    const int64_t slab0 = nslab * blockIdx.x / gridDim.x;
    const int64_t nmine = nslab * (blockIdx.x + 1) / gridDim.x - slab0;

    // Rounds: a round costs a full sequence of passes on its busiest sub-partition, i.e. ceil(slabs / 4)
    // slab-passes.  The split keeps the sum of those at its minimum ceil(n / 4) and, within that, the rounds
    // as even as possible: 28 slabs are 16 + 12 (4 + 3), 20 are 12 + 8, 17 are 9 + 8 -- not 16 + 4 or 16 + 1,
    // whose last round would leave most warps idle (b2f_round, also used by the complex kernel).
    const int64_t rounds = (nmine + C::NW * C::NGMAX - 1) / (C::NW * C::NGMAX);
    int64_t done = 0, units = (nmine + 3) >> 2;
    for (int64_t rd = 0; rd < rounds; ++rd) {
        const int64_t nround = b2f_round(nmine - done, rounds - rd, units);
        const int nact = (int)(nround < C::NW ? nround : C::NW);           // warps with work = ring members
        if (threadIdx.x == 0) {
            for (int i = 0; i < C::NS; ++i) {
                if (done > 0) {
                    mbar_inval(bar_full + 8 * i);
                    mbar_inval(bar_empty + 8 * i);
                }
                mbar_init(bar_full + 8 * i, 32);                           // 32 cp.async arrivals (one per lane)
                mbar_init(bar_empty + 8 * i, (uint32_t)nact);
            }
            mbar_fence_init();
        }
        __syncthreads();
        const int base = (int)(nround / C::NW), extra = (int)(nround % C::NW);
        const int ng = base + (warp < extra ? 1 : 0);
        const int64_t wslab0 = slab0 + done + (int64_t)warp * base + (warp < extra ? warp : extra);
        if (ng == 2)
            b2f_consume<2>(a, smem, lane, warp, warp, nact, wslab0 << 3);
        else if (ng == 1)
            b2f_consume<1>(a, smem, lane, warp, warp, nact, wslab0 << 3);
        done += nround;
        __syncthreads();                                                   // ring drained before it is re-initialised
    }
}

inline size_t b2f_scratch_bytes(int64_t N, int nbw)
{
    const int64_t Nv = (N - nbw - 1 > 0) ? N - nbw - 1 : 0;
    return (size_t)b2f_nblocks(Nv) * B2fCfg::NB * B2fCfg::NB * sizeof(double);
}

// launch plan: persistent grid, one CTA per SM, rounds of 16 slabs
inline int64_t b2f_grid(int64_t nev, int nsm)
{
    const int64_t nslab = (nev + 7) >> 3;
    return nslab < nsm ? nslab : nsm;
}

inline cudaError_t launch_b2f(int64_t N, int nbw, int64_t nev, const double *hv, int64_t ldv, const double *tau, double *q,
                              int64_t ldq, int align16, int nsm, void *scratch, cudaStream_t st)
{
    const int64_t Nv = N - nbw - 1;
    const int64_t npb = b2f_nblocks(Nv);
    double *tneg = (double *)scratch;
    b2f_tfactor_kernel<<<(unsigned)npb, 256, 0, st>>>(N, Nv, nbw, hv, ldv, tau, tneg);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if ((e = set_max_smem((const void *)bt_b2f_kernel, B2fCfg::SMEM_BYTES)) != cudaSuccess) return e;
    B2fArgs a;
    a.N = N;
    a.nev = nev;
    a.ldq = ldq;
    a.ldv = ldv;
    a.Nv = Nv;
    a.nbw = nbw;
    a.ew = 1;
    a.hv = hv;
    a.tneg = tneg;
    a.q = q;
    a.align16 = align16;
    bt_b2f_kernel<<<(unsigned)b2f_grid(nev, nsm), 256, B2fCfg::SMEM_BYTES, st>>>(a);
    return cudaGetLastError();
}

}  // namespace elpa2bt
