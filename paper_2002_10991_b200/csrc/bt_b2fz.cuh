// bt_b2fz.cuh -- band -> full back-transformation (Eq. 6e), COMPLEX FP64, on the FP64
// tensor cores (sm_100a).  Same algorithm, ring layout and fragment chaining as bt_b2f.cuh; every complex
// product is THREE real DMMAs (3M form) on planar register fragments, memory stays interleaved (re, im).
//
//      q <- H_0 H_1 ... H_{Nv-1} q,   H_j = I - tau_j v_j v_j^H  (R2: tau as stored, v^H in the dot)
//      blocks of 64: Q_p = I - V_p T_p V_p^H,  T upper triangular, T[i][i] = tau_i,
//                    T[:i, i] = -tau_i T[:i,:i] (V[:, :i]^H v_i)
//      W^T = q^T conj(V):  Wr += qr Vr + qi Vi,   Wi += qi Vr - qr Vi
//      U^T = W^T (-T)^T:   Ur = Wr Tr' - Wi Ti',  Ui = Wr Ti' + Wi Tr'      (T' = -T)
//      q^T += U^T V^T:     qr += Ur Vr - Ui Vi,   qi += Ur Vi + Ui Vr
//
// An interleaved complex N x Nv matrix is a real 2N x Nv matrix: the V ring (16 doubles = 8 complex rows
// x 64 reflectors per panel, reflector stride 18 doubles), the per-warp q ring and the tile stores are
// bt_b2f.cuh's, called with N, ldq, ldv counted in doubles.  With the stride of 18 doubles both
// B-fragment patterns (one LDS.128 = one complex element) are bank-conflict free:
//   update  B[k = r][n = gq] = V[row gq][reflector 8i+2r+e]   -> word offset 72 r + 4 gq = 8 r + 4 gq (mod 32)
//   dot     B[k = r][n = gq] = V[row 2r+e][reflector 8i+gq]   -> word offset 36 gq + 8 r   = 4 gq + 8 r (mod 32)
// Lane (gq, r) holds complex rows 2r, 2r+1 of column gq of an 8-row group (32 contiguous bytes).
// A warp owns ONE slab of 8 columns for all passes: the three accumulators of W (3M form, below) and U
// (5 x 16 doubles) live in registers.
#pragma once
#include "bt_b2f.cuh"

namespace elpa2bt {

// ---- prepass: -T_p of every block (plain FP64, complex) -------------------------------------------------
// One CTA (256 threads) per block p; dynamic shared memory B2FZ_TF_SMEM bytes.
constexpr int B2FZ_TF_SV = B2fCfg::NB + 1;
constexpr int B2FZ_TF_SMEM = (16 * B2FZ_TF_SV * 2 + B2fCfg::NB * B2FZ_TF_SV * 2 + 4 * B2fCfg::NB) * 8;

__global__ void __launch_bounds__(256) b2fz_tfactor_kernel(int64_t N, int64_t Nv, int nbw, const double *__restrict__ hv,
                                                           int64_t ldv, const double *__restrict__ tau,
                                                           double *__restrict__ tneg)
{
    constexpr int NB = B2fCfg::NB, RC = 16, SV = B2FZ_TF_SV;
    extern __shared__ __align__(16) double tf_smem[];
    double *Vs = tf_smem;                             // Vs[row][refl] (re, im)
    double *Sm = Vs + RC * SV * 2;                    // Gram matrix S = V^H V, then T (upper triangle)
    double *taus = Sm + NB * SV * 2;                  // (re, im)
    double *colS = taus + 2 * NB;
    const int tid = threadIdx.x;
    const int64_t p = blockIdx.x;
    const int64_t j0 = p * NB;
    const int nb = (int)((Nv - j0 < NB) ? Nv - j0 : NB);
    const int64_t i0 = j0 + nbw;
    const int ty = tid >> 4, tx = tid & 15;
    double accr[4][4], acci[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) accr[a][b] = acci[a][b] = 0.0;
    if (tid < NB) {
        taus[2 * tid] = (tid < nb) ? tau[2 * (j0 + tid)] : 0.0;
        taus[2 * tid + 1] = (tid < nb) ? tau[2 * (j0 + tid) + 1] : 0.0;
    }
    for (int64_t rb = i0; rb < N; rb += RC) {
        for (int idx = tid; idx < RC * NB; idx += 256) {
            const int c = idx >> 4, rr = idx & 15;
            const int64_t row = rb + rr;
            double2 v = make_double2(0.0, 0.0);
            if (c < nb && row < N) v = *reinterpret_cast<const double2 *>(hv + 2 * (row + (j0 + c) * ldv));
            *reinterpret_cast<double2 *>(Vs + 2 * (rr * SV + c)) = v;
        }
        __syncthreads();
#pragma unroll 2
        for (int rr = 0; rr < RC; ++rr) {
            double2 a4[4], b4[4];
#pragma unroll
            for (int a = 0; a < 4; ++a) a4[a] = *reinterpret_cast<const double2 *>(Vs + 2 * (rr * SV + 4 * ty + a));
#pragma unroll
            for (int b = 0; b < 4; ++b) b4[b] = *reinterpret_cast<const double2 *>(Vs + 2 * (rr * SV + 4 * tx + b));
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    // conj(a) * b
                    accr[a][b] = fma(a4[a].x, b4[b].x, accr[a][b]);
                    accr[a][b] = fma(a4[a].y, b4[b].y, accr[a][b]);
                    acci[a][b] = fma(a4[a].x, b4[b].y, acci[a][b]);
                    acci[a][b] = fma(-a4[a].y, b4[b].x, acci[a][b]);
                }
        }
        __syncthreads();
    }
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b)
            *reinterpret_cast<double2 *>(Sm + 2 * ((4 * ty + a) * SV + 4 * tx + b)) = make_double2(accr[a][b], acci[a][b]);
    __syncthreads();
    // larft (forward, columnwise), in place: thread r < i owns
    //   T[r][i] = -tau_i sum_{k = r}^{i-1} T[r][k] S[k][i]   (T[r][r] = tau_r; T[r][k], r < k < i, already final)
    for (int i = 0; i < NB; ++i) {
        if (tid < i) *reinterpret_cast<double2 *>(colS + 2 * tid) = *reinterpret_cast<const double2 *>(Sm + 2 * (tid * SV + i));
        __syncthreads();
        if (tid < i) {
            double sr = 0.0, si = 0.0;
            for (int k = tid; k < i; ++k) {
                const double tr = (k == tid) ? taus[2 * tid] : Sm[2 * (tid * SV + k)];
                const double ti = (k == tid) ? taus[2 * tid + 1] : Sm[2 * (tid * SV + k) + 1];
                const double cr = colS[2 * k], ci = colS[2 * k + 1];
                sr = fma(tr, cr, sr);
                sr = fma(-ti, ci, sr);
                si = fma(tr, ci, si);
                si = fma(ti, cr, si);
            }
            const double ur = taus[2 * i], ui = taus[2 * i + 1];
            Sm[2 * (tid * SV + i)] = -(ur * sr - ui * si);
            Sm[2 * (tid * SV + i) + 1] = -(ur * si + ui * sr);
        }
        __syncthreads();
    }
    // -T, row-major 64 x 64 interleaved, zeros below the diagonal
    double *out = tneg + p * (NB * NB * 2);
    for (int idx = tid; idx < NB * NB; idx += 256) {
        const int i = idx >> 6, k = idx & 63;
        double2 v = make_double2(0.0, 0.0);
        if (k > i)
            v = make_double2(-Sm[2 * (i * SV + k)], -Sm[2 * (i * SV + k) + 1]);
        else if (k == i)
            v = make_double2(-taus[2 * i], -taus[2 * i + 1]);
        *reinterpret_cast<double2 *>(out + 2 * idx) = v;
    }
}

// ---- a warp with one slab of 8 columns, all passes ------------------------------------------------------
__device__ __forceinline__ void b2fz_consume(const B2fArgs &a, unsigned char *smem, const int lane, const int warp,
                                             const int member, const int nmem, const int64_t col0)
{
    using C = B2fCfg;
    constexpr int NB = C::NB, S = C::S, NSP = C::NS, LAG = C::LAG, QS = C::QS, NSQ = C::NSQ, DQ = C::DQ;
    double *ring = reinterpret_cast<double *>(smem);
    double *qring = reinterpret_cast<double *>(smem + C::OFF_Q) + (size_t)warp * NSQ * C::QTILE;
    const uint32_t bar_full = smem_u32(smem + C::OFF_BAR);
    const uint32_t bar_empty = bar_full + C::NS * 8;
    const int gq = lane >> 2, r = lane & 3;
    const int64_t N = a.N;                              // doubles per column (2 x complex rows)
    const int64_t npb = b2f_nblocks(a.Nv);
    const int64_t ghi = (N - 1) >> 4;

    double *const cb = a.q + (col0 + gq < a.nev ? col0 + gq : 0) * a.ldq;
    const bool colok = col0 + gq < a.nev;
    const bool allcols = col0 + 8 <= a.nev;

    B2fCursor pc = {npb, b2f_glo(npb, a.nbw, 2)}, qc = pc;
    auto advance = [&](B2fCursor &c) {
        if (c.P < 0) return;
        if (c.g < ghi) {
            ++c.g;
        } else {
            --c.P;
            c.g = b2f_glo(c.P, a.nbw, 2);
        }
    };
    auto fetch_q = [&](int qst) {
        if (qc.P >= 0) b2f_fetch_q<1, 16>(a, qring + qst * C::QTILE, col0, qc.g, lane);
        cp_async_commit();                              // one group per item, empty past the end
        advance(qc);
    };
    uint32_t it = 0;
    int duty = 0, qst_in = 0, qst_out = 0;
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

    // n-tile i, entry e: reflector 8i + 2r + e of this lane's column
    // Both big products use the 3M form of a complex product (three real DMMAs instead of four; the operand
    // sums are one DADD each on the same FP64 pipe, 2 cycles against 16):
    //   dot:     P1 += qr Vr,  P2 += qi Vi,  P3 += (qr + qi)(Vr - Vi)   =>  Wr = P1 + P2,  Wi = P3 - P1 + P2
    //   update:  A = Ur Vr,    B = Ui Vi,    C = (Ur + Ui)(Vr + Vi)      =>  qr += A - B,   qi += C - A - B
    // P1..P3 are accumulated over a whole pass and turned into W at its end.
    double P1[8][2], P2[8][2], P3[8][2], Ur[8][2], Ui[8][2];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int e = 0; e < 2; ++e) P1[i][e] = P2[i][e] = P3[i][e] = Ur[i][e] = Ui[i][e] = 0.0;

    int64_t P = npb, g = b2f_glo(npb, a.nbw, 2);
    while (P >= 0) {
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
        fetch_q(qst_in);
        qst_in = (qst_in + 1 == NSQ) ? 0 : qst_in + 1;
        asm volatile("cp.async.wait_group %0;" ::"n"(DQ) : "memory");
        __syncwarp();
        const uint32_t st = it & (NSP - 1), ph = (it >> C::LGNS) & 1;
        mbar_wait(bar_full + 8 * st, ph);
        const double *pa = ring + st * C::STAGE_DOUBLES;      // V_P tile
        const double *pb = pa + C::PANEL;                     // V_{P-1} tile
        const bool has_upd = (P < npb) && ((g << 4) >= (P * NB + a.nbw) * 2);   // warp-uniform
        const bool has_dot = P >= 1;

        // complex rows 2r, 2r+1 of column gq
        double Yr[2], Yi[2];
        {
            const double *qt = qring + qst_out * C::QTILE + gq * QS + 4 * r;
            const double2 u = *reinterpret_cast<const double2 *>(qt);
            const double2 w = *reinterpret_cast<const double2 *>(qt + 2);
            Yr[0] = u.x, Yi[0] = u.y, Yr[1] = w.x, Yi[1] = w.y;
        }
        qst_out = (qst_out + 1 == NSQ) ? 0 : qst_out + 1;

        if (has_upd) {
            // --- q^T += U^T V_P^T: chunk (i, e): k-slot r = reflector 8i + 2r + e; A, B, C in two sets (e = 0 / 1):
            //     six independent accumulator chains
            double A[2][2] = {{0.0, 0.0}, {0.0, 0.0}}, B[2][2] = {{0.0, 0.0}, {0.0, 0.0}}, Cc[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
            const double *bp = pa + (2 * r) * S + 2 * gq;
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const double2 b = *reinterpret_cast<const double2 *>(bp + (8 * i + e) * S);
                    dmma884(A[e][0], A[e][1], Ur[i][e], b.x, A[e][0], A[e][1]);
                    dmma884(B[e][0], B[e][1], Ui[i][e], b.y, B[e][0], B[e][1]);
                    dmma884(Cc[e][0], Cc[e][1], Ur[i][e] + Ui[i][e], b.x + b.y, Cc[e][0], Cc[e][1]);
                }
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                const double pa_ = A[0][c] + A[1][c], pb_ = B[0][c] + B[1][c], pc_ = Cc[0][c] + Cc[1][c];
                Yr[c] += pa_ - pb_;
                Yi[c] += (pc_ - pa_) - pb_;
            }
        }
        if (has_dot) {
            // --- W^T += q^T conj(V_{P-1}): k-chunk e: k-slot r = row 2r + e; n-tile i = reflectors 8i + n
            const double Ys[2] = {Yr[0] + Yi[0], Yr[1] + Yi[1]};
            const double *bp = pb + gq * S + 4 * r;
#pragma unroll
            for (int i = 0; i < 8; i += 2) {
                double2 b[2][2];
#pragma unroll
                for (int d = 0; d < 2; ++d)
#pragma unroll
                    for (int e = 0; e < 2; ++e) b[d][e] = *reinterpret_cast<const double2 *>(bp + 8 * (i + d) * S + 2 * e);
#pragma unroll
                for (int e = 0; e < 2; ++e)
#pragma unroll
                    for (int d = 0; d < 2; ++d) {
                        dmma884(P1[i + d][0], P1[i + d][1], Yr[e], b[d][e].x, P1[i + d][0], P1[i + d][1]);
                        dmma884(P2[i + d][0], P2[i + d][1], Yi[e], b[d][e].y, P2[i + d][0], P2[i + d][1]);
                        dmma884(P3[i + d][0], P3[i + d][1], Ys[e], b[d][e].x - b[d][e].y, P3[i + d][0], P3[i + d][1]);
                    }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * st);
        if (has_upd) {
            const int64_t row = (g << 4) + 4 * r;
            const bool fast = allcols && ((g << 4) + 16 <= N);    // warp-uniform
            const double y[4] = {Yr[0], Yi[0], Yr[1], Yi[1]};
            b2f_store4(a, cb, colok, row, fast, y);
        }
        ++it;
        if (has_dot && g == ghi) {
            // --- end of pass: U^T = W^T (-T_{P-1})^T.  n-tile i' = reflectors 8i' + n; k chunk (i, e): k-slot r =
            //     reflector 8i + 2r + e; B[k][n] = T'[8i' + n][k], zero for k-tiles i < i' (T upper triangular)
            const double *tp = a.tneg + ((P - 1) * (NB * NB) + gq * NB + 2 * r) * 2;
            // W from the three accumulators, in place: Wr -> P1, Wi -> P3
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const double p1 = P1[i][e], p2 = P2[i][e];
                    P1[i][e] = p1 + p2;
                    P3[i][e] = (P3[i][e] - p1) + p2;
                }
#pragma unroll
            for (int ip = 0; ip < 8; ++ip) {
                double cr[2] = {0.0, 0.0}, ci[2] = {0.0, 0.0}, dr[2] = {0.0, 0.0}, di[2] = {0.0, 0.0};
#pragma unroll
                for (int i = ip; i < 8; ++i) {
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const double2 t = __ldg(reinterpret_cast<const double2 *>(tp + (8 * ip * NB + 8 * i + e) * 2));
                        dmma884(cr[0], cr[1], P1[i][e], t.x, cr[0], cr[1]);
                        dmma884(ci[0], ci[1], P1[i][e], t.y, ci[0], ci[1]);
                        dmma884(dr[0], dr[1], P3[i][e], -t.y, dr[0], dr[1]);
                        dmma884(di[0], di[1], P3[i][e], t.x, di[0], di[1]);
                    }
                }
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    Ur[ip][e] = cr[e] + dr[e];
                    Ui[ip][e] = ci[e] + di[e];
                }
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) P1[i][0] = P1[i][1] = P2[i][0] = P2[i][1] = P3[i][0] = P3[i][1] = 0.0;
        }
        if (g < ghi) {
            ++g;
        } else {
            --P;
            g = b2f_glo(P, a.nbw, 2);
        }
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
}

// ---- the kernel: CTA c takes slabs [nslab*c/grid, nslab*(c+1)/grid) in rounds of up to 8 (one per warp) ---
__global__ void __launch_bounds__(256, 1) bt_b2fz_kernel(const B2fArgs a)
{
    using C = B2fCfg;
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t bar_full = smem_u32(smem + C::OFF_BAR);
    const uint32_t bar_empty = bar_full + C::NS * 8;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t nslab = (a.nev + 7) >> 3;
    const int64_t slab0 = nslab * blockIdx.x / gridDim.x;
    const int64_t nmine = nslab * (blockIdx.x + 1) / gridDim.x - slab0;

    const int64_t rounds = (nmine + C::NW - 1) / C::NW;      // rounds sized by b2f_round (bt_b2f.cuh)
    int64_t done = 0, units = (nmine + 3) >> 2;
    for (int64_t rd = 0; rd < rounds; ++rd) {
        const int64_t nround = b2f_round(nmine - done, rounds - rd, units);
        const int nact = (int)nround;
        if (threadIdx.x == 0) {
            for (int i = 0; i < C::NS; ++i) {
                if (done > 0) {
                    mbar_inval(bar_full + 8 * i);
                    mbar_inval(bar_empty + 8 * i);
                }
                mbar_init(bar_full + 8 * i, 32);
                mbar_init(bar_empty + 8 * i, (uint32_t)nact);
            }
            mbar_fence_init();
        }
        __syncthreads();
        if (warp < nact) b2fz_consume(a, smem, lane, warp, warp, nact, (slab0 + done + warp) << 3);
        done += nround;
        __syncthreads();
    }
}

inline size_t b2fz_scratch_bytes(int64_t N, int nbw)
{
    const int64_t Nv = (N - nbw - 1 > 0) ? N - nbw - 1 : 0;
    return (size_t)b2f_nblocks(Nv) * B2fCfg::NB * B2fCfg::NB * 2 * sizeof(double);
}

// grid: as many CTAs as SMs x waves such that a CTA's rounds of 8 slabs are full when there is enough work
inline int64_t b2fz_grid(int64_t nev, int nsm)
{
    const int64_t nslab = (nev + 7) >> 3;
    return nslab < nsm ? nslab : nsm;
}

// hv, tau, q: interleaved complex; ldv, ldq in complex elements
inline cudaError_t launch_b2fz(int64_t N, int nbw, int64_t nev, const double *hv, int64_t ldv, const double *tau, double *q,
                               int64_t ldq, int nsm, void *scratch, cudaStream_t st)
{
    const int64_t Nv = N - nbw - 1;
    const int64_t npb = b2f_nblocks(Nv);
    double *tneg = (double *)scratch;
    cudaError_t e;
    if ((e = set_max_smem((const void *)b2fz_tfactor_kernel, B2FZ_TF_SMEM)) != cudaSuccess) return e;
    b2fz_tfactor_kernel<<<(unsigned)npb, 256, B2FZ_TF_SMEM, st>>>(N, Nv, nbw, hv, ldv, tau, tneg);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if ((e = set_max_smem((const void *)bt_b2fz_kernel, B2fCfg::SMEM_BYTES)) != cudaSuccess) return e;
    B2fArgs a;
    a.N = 2 * N;
    a.nev = nev;
    a.ldq = 2 * ldq;
    a.ldv = 2 * ldv;
    a.Nv = Nv;
    a.nbw = nbw;
    a.ew = 2;
    a.hv = hv;
    a.tneg = tneg;
    a.q = q;
    a.align16 = 1;
    bt_b2fz_kernel<<<(unsigned)b2fz_grid(nev, nsm), 256, B2fCfg::SMEM_BYTES, st>>>(a);
    return cudaGetLastError();
}

}  // namespace elpa2bt
