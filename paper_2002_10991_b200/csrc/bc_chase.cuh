// bc_chase.cuh -- SURVEY.md 8(f) NEXT-1, first version: bulge chasing of a real symmetric (and, further
// down, complex Hermitian) band matrix to tridiagonal form on the GPU (Eq. 6b), emitting the Householder reflectors
// directly in the device layout the back-transformation consumes (include/elpa2_bt.h).
//
// Step (s, k) -- sweep s, chase block k -- is exactly the oracle's step (R3, R7):
//   rows r0 = s+1+k nbw .. r1 = min(s+(k+1) nbw, N-1), eliminated column c = s (k = 0) or r0-nbw;
//   (v, tau, beta) from B[r0..r1][c]; B <- H^T B H on the three blocks that can be non-zero:
//   (i) B[r0..r1][c+1..r0-1], (ii) the diagonal block (symmetric rank-2 form), (iii) the block below.
// Parallelism: step (s+1, k) touches what steps (s+1, k-1), (s, k+1) and (s, k+2) wrote, but it shares
// only ONE element with (s, k+2): the latter's head element is the corner of the former's block (iii).
// Two schedules: a persistent kernel (one CTA per SM walks sweeps c, c+grid, ..; per-sweep "done" and
// "head" flags; dependency chain 2 steps per sweep) and, on request (ELPA2_BC_WAVEFRONT=1), one launch
// per wavefront t = 3s + k with stream order as the dependency.
// The band lives in global memory (L2-resident: (2 nbw + 1) N doubles); a CTA keeps v and the
// two work vectors of block (ii) in shared memory.  Every sum runs in the order SURVEY O3 / the oracle
// states and every product and sum is rounded separately (__dmul_rn / __dadd_rn: no FMA contraction):
// the tridiagonal form is unique but ill-conditioned (it is the Lanczos recurrence started at e1), so
// two backward-stable chases drift apart entry by entry as N grows; rounding exactly like the
// definition keeps the result reproducible and element-wise comparable at any N.
#pragma once
#include "bt_common.cuh"

namespace elpa2bt {

template <int NBW>
__device__ __forceinline__ void bc_step_global(const int64_t N, const int64_t s, const int64_t k, double *__restrict__ ab,
                                               double *__restrict__ hh_v, double *__restrict__ hh_tau, double *v, double *p,
                                               double *w2, double *red, double *sc, uint32_t *head_mine = nullptr,
                                               const uint32_t *head_prev = nullptr, const uint32_t need_head = 0,
                                               double *TD = nullptr)
{
    // TD != nullptr (persistent kernel, 384 threads): shared memory for the packed lower triangle of the
    // diagonal block + NBW dot products + the tile of block (i) (real: both fit, 196 KB at nbw = 128; block
    // (iii), whose accesses are coalesced anyway, stays in global memory); see bc_step_global_z
    constexpr int TRI = NBW * (NBW + 1) / 2;
    auto toff = [](int j) { return j * NBW - ((j * (j - 1)) >> 1); };
    constexpr int LG = (NBW == 32) ? 5 : (NBW == 64) ? 6 : 7;
    constexpr int64_t ldab = 2 * NBW + 1;
    const int tid = threadIdx.x, nt = blockDim.x;
    const int64_t r0 = s + 1 + (k << LG);
    int64_t r1 = s + ((k + 1) << LG);
    if (r1 > N - 1) r1 = N - 1;
    const int L = (int)(r1 - r0 + 1);
    const int64_t c = (k == 0) ? s : r0 - NBW;
    const int64_t g = hh_off(N, NBW, s) + k;
#define BC_B(i, j) ab[((i) - (j)) + (j) * ldab]
    double *vout = hh_v + g * NBW;
    if (k > 0 && L == 1) {                       // nothing to eliminate: identity slot (R3)
        for (int i = tid; i < NBW; i += nt) vout[i] = (i == 0) ? 1.0 : 0.0;
        if (tid == 0) {
            hh_tau[g] = 0.0;
            if (head_mine) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(head_mine), "r"((uint32_t)(k + 1)) : "memory");
        }
        return;
    }
    constexpr int LDA = NBW + 1;                       // column stride of the block (i) tile
    double *TA = TD ? TD + TRI + NBW : nullptr;        // block (i): column q = matrix column c+1+q, rows r0 ..
    if (TD) {
        for (int j = tid >> 5; j < L; j += nt >> 5) {
            const double *src = &BC_B(r0 + j, r0 + j);
            double *dst = TD + toff(j);
            for (int i = tid & 31; i < L - j; i += 32) cp_async8(smem_u32(dst + i), src + i, 8u);
        }
        for (int64_t j = c + 1 + (tid >> 5); j < r0; j += nt >> 5) {
            const double *src = &BC_B(r0, j);
            double *dst = TA + (j - (c + 1)) * LDA;
            for (int i = tid & 31; i < L; i += 32) cp_async8(smem_u32(dst + i), src + i, 8u);
        }
        cp_async_commit();
    }
    // --- Householder generator (R7): beta = -sign(alpha) ||x||, tau = (beta - alpha)/beta, v = x/(alpha - beta)
    if (tid < L) p[tid] = BC_B(r0 + tid, c);     // x, parked in p
    __syncthreads();
    if (tid == 0) {
        const double alpha = p[0];
        double ss = 0.0;
#pragma unroll 8
        for (int i = 1; i < L; ++i) ss = __dadd_rn(ss, __dmul_rn(p[i], p[i]));
        if (ss == 0.0) {
            sc[0] = 0.0;
            sc[1] = 0.0;
            sc[2] = alpha;
        } else {
            const double nrm = sqrt(__dadd_rn(__dmul_rn(alpha, alpha), ss));
            const double b = (alpha >= 0.0) ? -nrm : nrm;
            sc[0] = __ddiv_rn(__dsub_rn(b, alpha), b);
            sc[1] = __ddiv_rn(1.0, __dsub_rn(alpha, b));
            sc[2] = b;
        }
    }
    __syncthreads();
    const double tau = sc[0];
    for (int i = tid; i < NBW; i += nt) {
        const double vi = (i == 0) ? 1.0 : (i < L ? __dmul_rn(p[i], sc[1]) : 0.0);
        v[i] = vi;
        vout[i] = vi;
    }
    __syncthreads();
    if (tid < L) BC_B(r0 + tid, c) = (tid == 0) ? sc[2] : 0.0;
    if (tid == 0) {
        hh_tau[g] = tau;
        if (head_mine) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(head_mine), "r"((uint32_t)(k + 1)) : "memory");
    }
    if (TD) {
        cp_async_wait_all();
        __syncthreads();
    }
    if (tau == 0.0) return;
    if (TD) {
        const int grp = tid >> 7, t0 = tid & 127;
        double *dA = TD + TRI;
#define DD(i, j) (((i) >= (j)) ? TD[toff(j) + (i) - (j)] : TD[toff(i) + (j) - (i)])
        if (grp == 0) {
            for (int64_t j = c + 1 + t0; j < r0; j += 128) {
                const double *col = TA + (j - (c + 1)) * LDA;
                double dot = 0.0;
#pragma unroll 8
                for (int i = 0; i < L; ++i) dot = __dadd_rn(dot, __dmul_rn(v[i], col[i]));
                dA[j - (c + 1)] = dot;
            }
        } else if (grp == 1) {
            int64_t r2 = r1 + NBW;
            if (r2 > N - 1) r2 = N - 1;
            for (int64_t i = r1 + 1 + t0; i <= r2; i += 128) {
                if (need_head && i == r2) {      // the corner is the head element of step (s-1, k+2): wait for its beta
                    uint32_t h;
                    do {
                        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(h) : "l"(head_prev) : "memory");
                    } while (h < need_head);
                }
                // (batching these loads by hand, as in the complex step, was measured slower here: 1.42 s against 1.15 s)
                double dot = 0.0;
                for (int l = 0; l < L; ++l) dot = __dadd_rn(dot, __dmul_rn(BC_B(i, r0 + l), v[l]));
                for (int l = 0; l < L; ++l) BC_B(i, r0 + l) = __dsub_rn(BC_B(i, r0 + l), __dmul_rn(__dmul_rn(tau, dot), v[l]));
            }
        } else {
            for (int j = t0; j < L; j += 128) {
                double dot = 0.0;
#pragma unroll 8
                for (int i = 0; i < L; ++i) dot = __dadd_rn(dot, __dmul_rn(v[i], DD(i, j)));
                red[j] = dot;
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
            for (int i = t0; i < L; i += 128) {
                double dot = 0.0;
#pragma unroll 8
                for (int j = 0; j < L; ++j) {
                    const double m = __dsub_rn(DD(i, j), __dmul_rn(__dmul_rn(tau, v[i]), red[j]));
                    dot = __dadd_rn(dot, __dmul_rn(m, v[j]));
                }
                w2[i] = dot;
            }
        }
        __syncthreads();
        {
            const int ty = tid >> 7, i = tid & 127;
            if (i < L) {
                for (int64_t j = c + 1 + ty; j < r0; j += 3)
                    BC_B(r0 + i, j) = __dsub_rn(TA[(j - (c + 1)) * LDA + i], __dmul_rn(__dmul_rn(tau, v[i]), dA[j - (c + 1)]));
                for (int j = ty; j <= i; j += 3) {
                    const double m = __dsub_rn(TD[toff(j) + i - j], __dmul_rn(__dmul_rn(tau, v[i]), red[j]));
                    BC_B(r0 + i, r0 + j) = __dsub_rn(m, __dmul_rn(__dmul_rn(tau, w2[i]), v[j]));
                }
            }
        }
#undef DD
        return;
    }
    // 384 threads (persistent kernel): three groups of 128 run (i), (iii), (ii) side by side; see bc_step_global_z
    const bool par = nt >= 384;
    const int grp = par ? (tid >> 7) : 0, t0 = par ? (tid & 127) : tid, st_ = par ? 128 : nt;
    auto sync_ii = [&]() {
        if (par)
            asm volatile("bar.sync 1, 128;" ::: "memory");
        else
            __syncthreads();
    };
    if (!par || grp == 0) {
        // --- (i) A <- H^T A on the rest of the bulge block: one thread per column
        for (int64_t j = c + 1 + t0; j < r0; j += st_) {
            double dot = 0.0;
            for (int i = 0; i < L; ++i) dot = __dadd_rn(dot, __dmul_rn(v[i], BC_B(r0 + i, j)));
            for (int i = 0; i < L; ++i) BC_B(r0 + i, j) = __dsub_rn(BC_B(r0 + i, j), __dmul_rn(__dmul_rn(tau, v[i]), dot));
        }
    }
    if (!par || grp == 2) {
        // --- (ii) D <- H^T D H: red = D v;  M = D - tau v red^T;  w2 = M v;  D' = M - tau w2 v^T (lower part)
        for (int j = t0; j < L; j += st_) {
            double dot = 0.0;
            for (int i = 0; i < L; ++i)
                dot = __dadd_rn(dot, __dmul_rn(v[i], (i >= j) ? BC_B(r0 + i, r0 + j) : BC_B(r0 + j, r0 + i)));
            red[j] = dot;
        }
        sync_ii();
        for (int i = t0; i < L; i += st_) {
            double dot = 0.0;
            for (int j = 0; j < L; ++j) {
                const double dij = (i >= j) ? BC_B(r0 + i, r0 + j) : BC_B(r0 + j, r0 + i);
                const double m = __dsub_rn(dij, __dmul_rn(__dmul_rn(tau, v[i]), red[j]));
                dot = __dadd_rn(dot, __dmul_rn(m, v[j]));
            }
            w2[i] = dot;
        }
        sync_ii();
        for (int j = t0; j < L; j += st_)
            for (int i = j; i < L; ++i) {
                const double m = __dsub_rn(BC_B(r0 + i, r0 + j), __dmul_rn(__dmul_rn(tau, v[i]), red[j]));
                BC_B(r0 + i, r0 + j) = __dsub_rn(m, __dmul_rn(__dmul_rn(tau, w2[i]), v[j]));
            }
    }
    if (!par || grp == 1) {
        // --- (iii) E <- E H on the block below: one thread per row; creates the next bulge
        int64_t r2 = r1 + NBW;
        if (r2 > N - 1) r2 = N - 1;
        for (int64_t i = r1 + 1 + t0; i <= r2; i += st_) {
            if (need_head && i == r2) {          // the corner is the head element of step (s-1, k+2): wait for its beta
                uint32_t h;
                do {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(h) : "l"(head_prev) : "memory");
                } while (h < need_head);
            }
            double dot = 0.0;
            for (int l = 0; l < L; ++l) dot = __dadd_rn(dot, __dmul_rn(BC_B(i, r0 + l), v[l]));
            for (int l = 0; l < L; ++l) BC_B(i, r0 + l) = __dsub_rn(BC_B(i, r0 + l), __dmul_rn(__dmul_rn(tau, dot), v[l]));
        }
    }
#undef BC_B
}

template <int NBW>
__global__ void __launch_bounds__(128) bc_wavefront_kernel(int64_t N, int64_t t, int64_t s_hi, double *__restrict__ ab,
                                                           double *__restrict__ hh_v, double *__restrict__ hh_tau)
{
    constexpr int LG = (NBW == 32) ? 5 : (NBW == 64) ? 6 : 7;
    __shared__ double v[NBW], p[NBW], w2[NBW], red[128], sc[3];
    const int64_t s = s_hi - blockIdx.x;
    if (s < 0) return;
    const int64_t k = t - 3 * s;
    const int64_t K = (N - 1 - s + NBW - 1) >> LG;
    if (k < 0 || k >= K) return;
    bc_step_global<NBW>(N, s, k, ab, hh_v, hh_tau, v, p, w2, red, sc);
}

// persistent version of the nbw = 128 step (block (ii) and, real, block (i) in shared memory; see TD in
// bc_step_global): flags and 2-step lag as in
// bc_persistent_kernel below
template <int NBW>
__global__ void __launch_bounds__(384) bc_persistent_global_kernel(int64_t N, double *__restrict__ ab,
                                                                   double *__restrict__ hh_v, double *__restrict__ hh_tau,
                                                                   uint32_t *__restrict__ prog)
{
    constexpr int LG = (NBW == 32) ? 5 : (NBW == 64) ? 6 : 7;
    extern __shared__ double td_smem[];                // packed triangle of the diagonal block + NBW dots
    __shared__ double v[NBW], p[NBW], w2[NBW], red[128], sc[3];
    const int tid = threadIdx.x;
    uint32_t *done = prog, *head = prog + N;
    for (int64_t s = blockIdx.x; s <= N - 2; s += gridDim.x) {
        const int64_t K = (N - 1 - s + NBW - 1) >> LG;
        const int64_t Kprev = (N - s + NBW - 1) >> LG;
        uint32_t known = 0;
        for (int64_t k = 0; k < K; ++k) {
            uint32_t need_head = 0;
            if (s > 0) {
                const uint32_t need = (uint32_t)((k + 2 < Kprev) ? k + 2 : Kprev);
                if (tid == 0) {
                    while (known < need) {
                        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(known) : "l"(done + s - 1) : "memory");
                    }
                }
                __syncthreads();
                if (k + 2 < Kprev) need_head = (uint32_t)(k + 3);
            }
            bc_step_global<NBW>(N, s, k, ab, hh_v, hh_tau, v, p, w2, red, sc, head + s, head + s - 1, need_head, td_smem);
            // the CTA barrier orders every thread's stores before thread 0's release (the pattern grid-wide
            // barriers are built from): one fence, not one per thread
            __syncthreads();
            if (tid == 0) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(done + s), "r"((uint32_t)(k + 1)) : "memory");
        }
    }
}

// ---- the same step with its three blocks staged in shared memory (nbw <= 64) -------------------------
// In band storage every column j of the step's region is ONE contiguous segment: rows r0..r1 for
// c < j < r0 (block i), rows j..r2 for r0 <= j <= r1 (lower part of block ii + block iii).  The CTA
// copies those segments into a tile S[col][row - r0] (column stride odd: conflict-free both ways),
// runs the step there with exactly the arithmetic of bc_wavefront_kernel, and copies them back.
template <int NBW>
__device__ __forceinline__ bool bc_step_smem(const int64_t N, const int64_t s, const int64_t k, double *__restrict__ ab,
                                             double *__restrict__ hh_v, double *__restrict__ hh_tau, double *S, double *v,
                                             double *p, double *w2, double *sc, uint32_t *head_mine = nullptr,
                                             const uint32_t *head_prev = nullptr, const uint32_t need_head = 0,
                                             const bool e_in = false, const bool allow_keep = false)
{
    // e_in: the previous step of this sweep left its block (iii) in S instead of writing it back -- it is
    // this step's column x and block (i).  Returns true if this step does the same for the next one
    // (allow_keep, persistent kernel only).  No other sweep reads that block in between: sweep s+1 needs
    // it only after the next step has written it out, sweep s-1 shares just the corner, see below.
    constexpr int LG = (NBW == 32) ? 5 : 6;
    constexpr int64_t ldab = 2 * NBW + 1;
    constexpr int LDS = 2 * NBW + 1;              // tile column stride (doubles)
    const int tid = threadIdx.x, nt = blockDim.x;
    const int64_t r0 = s + 1 + (k << LG);
    int64_t r1 = s + ((k + 1) << LG);
    if (r1 > N - 1) r1 = N - 1;
    const int L = (int)(r1 - r0 + 1);
    const int64_t c = (k == 0) ? s : r0 - NBW;
    const int64_t g = hh_off(N, NBW, s) + k;
    double *vout = hh_v + g * NBW;
    if (k > 0 && L == 1) {
        for (int i = tid; i < NBW; i += nt) vout[i] = (i == 0) ? 1.0 : 0.0;
        if (tid == 0) {
            hh_tau[g] = 0.0;
            if (head_mine) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(head_mine), "r"((uint32_t)(k + 1)) : "memory");
        }
        return false;
    }
    int64_t r2 = r1 + NBW;
    if (r2 > N - 1) r2 = N - 1;
    const int nA = (int)(r0 - c - 1);             // columns of block (i): c+1 .. r0-1
    const int nR = (int)(r2 - r0 + 1);            // tile rows: r0 .. r2
    const int ncol = nA + L;                      // tile columns: c+1 .. r1
    // tile column q <-> matrix column c+1+q; element (row, col) at S[q * LDS + row - r0]
    auto seg = [&](int q, int &lo, int &hi) {     // local rows [lo, hi) stored for tile column q
        if (q < nA) {
            lo = 0;
            hi = L;
        } else {
            lo = q - nA;
            hi = nR;
        }
    };
    // the next step's L is nR - L: keep block (iii) in S for it unless it is a one-row identity slot
    const bool keep = allow_keep && (nR - L >= 2);
    const int warp = tid >> 5, lane = tid & 31, nwarp = nt >> 5;
    int qs = 0;                                   // first tile column to fetch from global memory
    if (e_in) {
        // previous step: L = NBW, its block (iii) sits at columns nAp .. nAp+NBW-1, rows NBW .. NBW+L-1
        constexpr int MV = ((NBW - 1) * NBW + 255) / 256;
        const int nAp = (k == 1) ? 0 : NBW - 1;
        double tmp[MV];
#pragma unroll
        for (int m = 0; m < MV; ++m) {
            const int idx = tid + m * 256, q = idx >> LG, row = idx & (NBW - 1);
            tmp[m] = (q < NBW - 1 && row < L) ? S[(nAp + 1 + q) * LDS + NBW + row] : 0.0;
        }
        if (tid < L) p[tid] = S[nAp * LDS + NBW + tid];        // x = its first column
        __syncthreads();
#pragma unroll
        for (int m = 0; m < MV; ++m) {
            const int idx = tid + m * 256, q = idx >> LG, row = idx & (NBW - 1);
            if (q < NBW - 1 && row < L) S[q * LDS + row] = tmp[m];
        }
        qs = nA;
    }
    // --- stage in: a warp per column, lanes along the column's contiguous band segment; cp.async keeps
    //     every copy in flight at once
    for (int q = qs + warp; q < ncol; q += nwarp) {
        int lo, hi;
        seg(q, lo, hi);
        const int64_t j = c + 1 + q;
        const double *src = ab + (r0 - j) + j * ldab;          // element (r0 + row, j) at src[row]
        double *dst = S + q * LDS;
        for (int row = lo + lane; row < hi; row += 32) cp_async8(smem_u32(dst + row), src + row, 8u);
    }
    cp_async_commit();
    if (!e_in && tid < L) p[tid] = ab[(r0 + tid - c) + c * ldab];       // x = B[r0..r1][c]
    cp_async_wait_all();
    __syncthreads();
#define BS(rl, q) S[(q) * LDS + (rl)]
    if (tid == 0) {
        const double alpha = p[0];
        double ss = 0.0;
#pragma unroll 8
        for (int i = 1; i < L; ++i) ss = __dadd_rn(ss, __dmul_rn(p[i], p[i]));
        if (ss == 0.0) {
            sc[0] = 0.0;
            sc[1] = 0.0;
            sc[2] = alpha;
        } else {
            const double nrm = sqrt(__dadd_rn(__dmul_rn(alpha, alpha), ss));
            const double b = (alpha >= 0.0) ? -nrm : nrm;
            sc[0] = __ddiv_rn(__dsub_rn(b, alpha), b);
            sc[1] = __ddiv_rn(1.0, __dsub_rn(alpha, b));
            sc[2] = b;
        }
    }
    __syncthreads();
    const double tau = sc[0];
    for (int i = tid; i < NBW; i += nt) {
        const double vi = (i == 0) ? 1.0 : (i < L ? __dmul_rn(p[i], sc[1]) : 0.0);
        v[i] = vi;
        vout[i] = vi;
    }
    if (tid < L) ab[(r0 + tid - c) + c * ldab] = (tid == 0) ? sc[2] : 0.0;
    if (tid == 0) {
        hh_tau[g] = tau;
        // persistent mode: the head element (beta) is all the next sweep's step (s+1, k-2) still lacks
        if (head_mine) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(head_mine), "r"((uint32_t)(k + 1)) : "memory");
    }
    __syncthreads();
    if (tau == 0.0 && !e_in) return false;        // the tile is unchanged and all of it is in global memory
    // Blocks (i), (ii), (iii) are disjoint and only read v: three groups of 64 threads run them side by
    // side; the two internal barriers of (ii) are named barriers of its own 64 threads.
    const int grp = (tau == 0.0) ? 3 : (tid >> 6), t64 = tid & 63;
    if (grp == 3) {
        // identity step that goes on because it holds the previous step's block (iii): nothing to compute,
        // but the corner staged in above may predate the beta of step (s-1, k+2) -- it must not be staged
        // out (or handed on) stale.  Same wait and re-fetch as group 1 below.
        if (need_head && tid == 0 && nR > L) {
            uint32_t h;
            do {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(h) : "l"(head_prev) : "memory");
            } while (h < need_head);
            const int64_t jc = c + 1 + (nA + L - 1);
            BS(nR - 1, nA + L - 1) = __ldcg(&ab[(r0 + nR - 1 - jc) + jc * ldab]);
        }
    } else if (grp == 0) {
        // --- (i): one thread per column q < nA
        for (int q = t64; q < nA; q += 64) {
            double dot = 0.0;
#pragma unroll 8
            for (int i = 0; i < L; ++i) dot = __dadd_rn(dot, __dmul_rn(v[i], BS(i, q)));
#pragma unroll 8
            for (int i = 0; i < L; ++i) BS(i, q) = __dsub_rn(BS(i, q), __dmul_rn(__dmul_rn(tau, v[i]), dot));
        }
    } else if (grp == 1) {
        // --- (iii): one thread per row L .. nR-1
        for (int rl = L + t64; rl < nR; rl += 64) {
            if (need_head && rl == nR - 1) {
                // the corner (last row, last column) is the head element of step (s-1, k+2), which may be
                // running right now: wait until it has written beta there, then fetch it
                uint32_t h;
                do {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(h) : "l"(head_prev) : "memory");
                } while (h < need_head);
                const int64_t jc = c + 1 + (nA + L - 1);
                BS(rl, nA + L - 1) = __ldcg(&ab[(r0 + rl - jc) + jc * ldab]);
            }
            double dot = 0.0;
#pragma unroll 8
            for (int l = 0; l < L; ++l) dot = __dadd_rn(dot, __dmul_rn(BS(rl, nA + l), v[l]));
#pragma unroll 8
            for (int l = 0; l < L; ++l)
                BS(rl, nA + l) = __dsub_rn(BS(rl, nA + l), __dmul_rn(__dmul_rn(tau, dot), v[l]));
        }
    } else if (grp == 2) {
        // --- (ii): D(i, j) = BS(max, nA + min);  p = D v;  M = D - tau v p^T;  w2 = M v;  D' = M - tau w2 v^T
        for (int j = t64; j < L; j += 64) {
            double dot = 0.0;
#pragma unroll 8
            for (int i = 0; i < L; ++i) dot = __dadd_rn(dot, __dmul_rn(v[i], (i >= j) ? BS(i, nA + j) : BS(j, nA + i)));
            p[j] = dot;
        }
        asm volatile("bar.sync 1, 64;" ::: "memory");
        for (int i = t64; i < L; i += 64) {
            double dot = 0.0;
#pragma unroll 8
            for (int j = 0; j < L; ++j) {
                const double dij = (i >= j) ? BS(i, nA + j) : BS(j, nA + i);
                const double m = __dsub_rn(dij, __dmul_rn(__dmul_rn(tau, v[i]), p[j]));
                dot = __dadd_rn(dot, __dmul_rn(m, v[j]));
            }
            w2[i] = dot;
        }
    }
    __syncthreads();
    // (ii), last phase: D' = M - tau w2 v^T is element-wise -- all threads (its owner group alone, one thread per
    // column with up to L elements each, was the longest chain of the step)
    if (tau != 0.0) {
        const int ty = tid / NBW, i = tid - ty * NBW, RY = nt / NBW;
        for (int j = ty; j < L; j += RY)
            if (i >= j && i < L) {
                const double m = __dsub_rn(BS(i, nA + j), __dmul_rn(__dmul_rn(tau, v[i]), p[j]));
                BS(i, nA + j) = __dsub_rn(m, __dmul_rn(__dmul_rn(tau, w2[i]), v[j]));
            }
        __syncthreads();
    }
#undef BS
    // --- stage out (block (iii) stays behind if the next step takes it from S): a warp per column, two
    //     columns at a time through registers, so that the shared-memory loads of both are in flight together
    //     (the one-column loop spent 5.3 k of the step's 24 k cycles here, this form 2.3 k)
    for (int q = warp; q < ncol; q += 2 * nwarp) {
        double t0[4], t1[4];
        int lo0, hi0, lo1 = 0, hi1 = 0;
        seg(q, lo0, hi0);
        if (keep && q >= nA) hi0 = L;
        const int q1 = q + nwarp;
        if (q1 < ncol) {
            seg(q1, lo1, hi1);
            if (keep && q1 >= nA) hi1 = L;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int ra = lo0 + lane + 32 * u, rb = lo1 + lane + 32 * u;
            if (ra < hi0) t0[u] = S[q * LDS + ra];
            if (rb < hi1) t1[u] = S[q1 * LDS + rb];
        }
        const int64_t j0 = c + 1 + q, j1 = c + 1 + q1;
        double *d0 = ab + (r0 - j0) + j0 * ldab, *d1 = ab + (r0 - j1) + j1 * ldab;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int ra = lo0 + lane + 32 * u, rb = lo1 + lane + 32 * u;
            if (ra < hi0) d0[ra] = t0[u];
            if (rb < hi1) d1[rb] = t1[u];
        }
    }
    return keep;
}

// one launch per wavefront t = 3s + k
template <int NBW>
__global__ void __launch_bounds__(256) bc_wavefront_smem_kernel(int64_t N, int64_t t, int64_t s_hi,
                                                                double *__restrict__ ab, double *__restrict__ hh_v,
                                                                double *__restrict__ hh_tau)
{
    constexpr int LG = (NBW == 32) ? 5 : 6;
    extern __shared__ double S[];                 // (2 NBW - 1) columns x (2 NBW + 1)
    __shared__ double v[NBW], p[NBW], w2[NBW], sc[3];
    const int64_t s = s_hi - blockIdx.x;
    if (s < 0) return;
    const int64_t k = t - 3 * s;
    const int64_t K = (N - 1 - s + NBW - 1) >> LG;
    if (k < 0 || k >= K) return;
    bc_step_smem<NBW>(N, s, k, ab, hh_v, hh_tau, S, v, p, w2, sc);
}

// persistent version: one CTA per SM, CTA c walks sweeps c, c + grid, ...  Step (s, k) overlaps step
// (s-1, k+2) in ONE element only -- the head element of (s-1, k+2) is the corner (last row, last column)
// of (s, k)'s block below -- so (s, k) starts as soon as (s-1, k+1) is finished (done[s-1] >= k+2) and
// only the thread that owns the last row of the block below waits for head[s-1] >= k+3, i.e. for
// (s-1, k+2) to have written its beta (which it does first thing, after reading the old value: no
// write-after-read hazard either).  The dependency chain is 2 steps per sweep instead of 3.  Flags are
// published with gpu-scope releases after the stores they cover and polled with gpu-scope acquires
// (which also drop the SM's L1 lines, so the staging copies read what the other SM wrote).
template <int NBW>
__global__ void __launch_bounds__(256) bc_persistent_kernel(int64_t N, double *__restrict__ ab, double *__restrict__ hh_v,
                                                            double *__restrict__ hh_tau, uint32_t *__restrict__ prog)
{
    constexpr int LG = (NBW == 32) ? 5 : 6;
    extern __shared__ double S[];
    __shared__ double v[NBW], p[NBW], w2[NBW], sc[3];
    const int tid = threadIdx.x;
    uint32_t *done = prog, *head = prog + N;          // steps finished / steps whose head element is written
    for (int64_t s = blockIdx.x; s <= N - 2; s += gridDim.x) {
        const int64_t K = (N - 1 - s + NBW - 1) >> LG;
        const int64_t Kprev = (N - s + NBW - 1) >> LG;      // K(s-1)
        uint32_t known = 0;
        bool e_in = false;                              // block (iii) of the previous step is still in S
        for (int64_t k = 0; k < K; ++k) {
            uint32_t need_head = 0;
            if (s > 0) {
                // everything but the corner of the block below: step (s-1, k+1) finished
                const uint32_t need = (uint32_t)((k + 2 < Kprev) ? k + 2 : Kprev);
                if (tid == 0) {
                    while (known < need) {
                        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(known) : "l"(done + s - 1) : "memory");
                    }
                }
                __syncthreads();
                if (k + 2 < Kprev) need_head = (uint32_t)(k + 3);    // step (s-1, k+2) exists: its beta is our corner
            }
            e_in = bc_step_smem<NBW>(N, s, k, ab, hh_v, hh_tau, S, v, p, w2, sc, head + s, head + s - 1, need_head, e_in, true);
            // the CTA barrier orders every thread's stores before thread 0's release (the pattern grid-wide
            // barriers are built from): one fence, not one per thread
            __syncthreads();
            if (tid == 0) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(done + s), "r"((uint32_t)(k + 1)) : "memory");
        }
    }
}

// ---- complex Hermitian version (global-memory step; the tile of a complex step exceeds shared memory) ----
// Complex arithmetic rounded like C99 without contraction (what the definition's plain loops mean and
// what the oracle's compiler emits): (a+bi)(c+di) = (ac - bd) + (ad + bc)i with four separately rounded
// products; 1/(c+di) by Smith's formula, the one libgcc's __divdc3 evaluates for in-range operands.
struct zc {
    double re, im;
};
__device__ __forceinline__ zc zmul(zc a, zc b)
{
    return {__dsub_rn(__dmul_rn(a.re, b.re), __dmul_rn(a.im, b.im)), __dadd_rn(__dmul_rn(a.re, b.im), __dmul_rn(a.im, b.re))};
}
__device__ __forceinline__ zc zadd(zc a, zc b) { return {__dadd_rn(a.re, b.re), __dadd_rn(a.im, b.im)}; }
__device__ __forceinline__ zc zsub(zc a, zc b) { return {__dsub_rn(a.re, b.re), __dsub_rn(a.im, b.im)}; }
__device__ __forceinline__ zc zconj(zc a) { return {a.re, -a.im}; }
__device__ __forceinline__ zc zrecip(zc z)        // 1 / z
{
    const double c = z.re, d = z.im;
    if (fabs(c) < fabs(d)) {
        const double ratio = __ddiv_rn(c, d), denom = __dadd_rn(__dmul_rn(c, ratio), d);
        return {__ddiv_rn(ratio, denom), __ddiv_rn(-1.0, denom)};
    }
    const double ratio = __ddiv_rn(d, c), denom = __dadd_rn(__dmul_rn(d, ratio), c);
    return {__ddiv_rn(1.0, denom), __ddiv_rn(-ratio, denom)};
}

template <int NBW>
__device__ __forceinline__ void bc_step_global_z(const int64_t N, const int64_t s, const int64_t k, zc *__restrict__ ab,
                                                 zc *__restrict__ hh_v, zc *__restrict__ hh_tau, zc *v, zc *p, zc *w2,
                                                 zc *zsc, double *dsc, uint32_t *head_mine = nullptr,
                                                 const uint32_t *head_prev = nullptr, const uint32_t need_head = 0,
                                                 zc *TD = nullptr)
{
    // TD != nullptr (persistent kernel, 384 threads): shared memory for the lower triangle of the diagonal
    // block, packed by columns (column j: rows j .. NBW-1 at TD + toff(j)), followed by NBW dot products.
    // Block (ii) -- three dependent phases, the longest chain of the step -- then runs out of shared
    // memory, and the element-wise second halves of (i) and (ii) run on all threads with coalesced
    // accesses after the groups have met.  Same operations in the same order within every sum.
    constexpr int TRI = NBW * (NBW + 1) / 2;
    auto toff = [](int j) { return j * NBW - ((j * (j - 1)) >> 1); };
    constexpr int LG = (NBW == 32) ? 5 : (NBW == 64) ? 6 : 7;
    constexpr int64_t ldab = 2 * NBW + 1;
    const int tid = threadIdx.x, nt = blockDim.x;
    const int64_t r0 = s + 1 + (k << LG);
    int64_t r1 = s + ((k + 1) << LG);
    if (r1 > N - 1) r1 = N - 1;
    const int L = (int)(r1 - r0 + 1);
    const int64_t c = (k == 0) ? s : r0 - NBW;
    const int64_t g = hh_off(N, NBW, s) + k;
#define BC_Z(i, j) ab[((i) - (j)) + (j) * ldab]
    zc *vout = hh_v + g * NBW;
    if (k > 0 && L == 1) {
        for (int i = tid; i < NBW; i += nt) vout[i] = {(i == 0) ? 1.0 : 0.0, 0.0};
        if (tid == 0) {
            hh_tau[g] = {0.0, 0.0};
            if (head_mine) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(head_mine), "r"((uint32_t)(k + 1)) : "memory");
        }
        return;
    }
    if (TD) {
        // the diagonal block was last written by steps that are finished (done flags): fetch it while the
        // generator runs; a warp per column, lanes along its contiguous rows
        for (int j = tid >> 5; j < L; j += nt >> 5) {
            const zc *src = &BC_Z(r0 + j, r0 + j);
            zc *dst = TD + toff(j);
            for (int i = tid & 31; i < L - j; i += 32) cp_async16(smem_u32(dst + i), src + i, 16u);
        }
        cp_async_commit();
    }
    // --- Householder generator (R2, R7): beta real, tau = ((beta - Re a)/beta, -Im a/beta), v = x/(alpha - beta)
    if (tid < L) p[tid] = BC_Z(r0 + tid, c);
    __syncthreads();
    if (tid == 0) {
        const double ar = p[0].re, ai = p[0].im;
        double ss = 0.0;
        for (int i = 1; i < L; ++i) ss = __dadd_rn(ss, __dadd_rn(__dmul_rn(p[i].re, p[i].re), __dmul_rn(p[i].im, p[i].im)));
        if (ss == 0.0 && ai == 0.0) {
            zsc[0] = {0.0, 0.0};
            zsc[1] = {0.0, 0.0};
            dsc[0] = ar;
        } else {
            const double nrm = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(ar, ar), __dmul_rn(ai, ai)), ss));
            const double b = (ar >= 0.0) ? -nrm : nrm;
            zsc[0] = {__ddiv_rn(__dsub_rn(b, ar), b), __ddiv_rn(-ai, b)};
            zsc[1] = zrecip({__dsub_rn(ar, b), ai});
            dsc[0] = b;
        }
    }
    __syncthreads();
    const zc tau = zsc[0], ctau = zconj(zsc[0]);
    const bool ident = (tau.re == 0.0 && tau.im == 0.0);
    for (int i = tid; i < NBW; i += nt) {
        zc vi = {0.0, 0.0};
        if (i == 0) vi = {1.0, 0.0};
        else if (i < L && !ident) vi = zmul(p[i], zsc[1]);
        v[i] = vi;
        vout[i] = vi;
    }
    __syncthreads();
    if (tid < L) BC_Z(r0 + tid, c) = {(tid == 0) ? dsc[0] : 0.0, 0.0};
    if (tid == 0) {
        hh_tau[g] = tau;
        if (head_mine) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(head_mine), "r"((uint32_t)(k + 1)) : "memory");
    }
    if (TD) {
        cp_async_wait_all();
        __syncthreads();
    }
    if (ident) return;
    if (TD) {
        const int grp = tid >> 7, t0 = tid & 127;
        zc *dA = TD + TRI;
#define DZ(i, j) (((i) >= (j)) ? TD[toff(j) + (i) - (j)] : zconj(TD[toff(i) + (j) - (i)]))
        if (grp == 0) {
            // --- (i), first half: the dot products v^H A, one thread per column.  The block (260 KB) does not fit
            //     beside the triangle, so it passes through shared memory 16 rows at a time (two buffers,
            //     [column][17 elements]): the copies are coalesced (16 lanes along the 256 contiguous bytes of
            //     a column) and the next chunk is in flight while this one is summed, in the definition's order
            const int nA = (int)(r0 - c - 1);
            if (nA > 0) {
                zc *CH = TD + TRI + NBW;
                constexpr int CS = 17, CB = (NBW - 1) * CS;
                const int nch = (L + 15) >> 4;
                auto fetch = [&](int ch, int buf) {
                    const int i = 16 * ch + (t0 & 15);
                    for (int q = t0 >> 4; q < nA; q += 8)
                        cp_async16(smem_u32(CH + buf * CB + q * CS + (t0 & 15)), &BC_Z(r0 + (i < L ? i : 0), c + 1 + q),
                                   i < L ? 16u : 0u);
                    cp_async_commit();
                };
                fetch(0, 0);
                zc dot = {0.0, 0.0};
                for (int ch = 0; ch < nch; ++ch) {
                    if (ch + 1 < nch) {
                        fetch(ch + 1, (ch + 1) & 1);
                        asm volatile("cp.async.wait_group 1;" ::: "memory");
                    } else {
                        asm volatile("cp.async.wait_group 0;" ::: "memory");
                    }
                    asm volatile("bar.sync 2, 128;" ::: "memory");
                    if (t0 < nA) {
                        const zc *col = CH + (ch & 1) * CB + t0 * CS;
#pragma unroll
                        for (int r = 0; r < 16; ++r)
                            if (16 * ch + r < L) dot = zadd(dot, zmul(zconj(v[16 * ch + r]), col[r]));
                    }
                    asm volatile("bar.sync 2, 128;" ::: "memory");      // the buffer may be refilled
                }
                if (t0 < nA) dA[t0] = dot;
            }
        } else if (grp == 1) {
            // --- (iii) E <- E H = E - tau (E v) v^H, one thread per row (coalesced both ways)
            int64_t r2 = r1 + NBW;
            if (r2 > N - 1) r2 = N - 1;
            for (int64_t i = r1 + 1 + t0; i <= r2; i += 128) {
                if (need_head && i == r2) {      // the corner is the head element of step (s-1, k+2): wait for its beta
                    uint32_t h;
                    do {
                        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(h) : "l"(head_prev) : "memory");
                    } while (h < need_head);
                }
                // (eight loads in flight at a time -- the row's elements are 4 KB apart; the sum keeps its order)
                zc dot = {0.0, 0.0};
                for (int l0 = 0; l0 < L; l0 += 8) {
                    zc e[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if (l0 + u < L) e[u] = BC_Z(i, r0 + l0 + u);
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if (l0 + u < L) dot = zadd(dot, zmul(e[u], v[l0 + u]));
                }
                const zc td = zmul(tau, dot);
                for (int l0 = 0; l0 < L; l0 += 8) {
                    zc e[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if (l0 + u < L) e[u] = BC_Z(i, r0 + l0 + u);
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if (l0 + u < L) BC_Z(i, r0 + l0 + u) = zsub(e[u], zmul(td, zconj(v[l0 + u])));
                }
            }
        } else {
            // --- (ii), first two phases, out of shared memory: p = v^H D;  w2 = (D - conj(tau) v p) v
            for (int j = t0; j < L; j += 128) {
                zc dot = {0.0, 0.0};
#pragma unroll 4
                for (int i = 0; i < L; ++i) dot = zadd(dot, zmul(zconj(v[i]), DZ(i, j)));
                p[j] = dot;
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
            for (int i = t0; i < L; i += 128) {
                zc dot = {0.0, 0.0};
#pragma unroll 4
                for (int j = 0; j < L; ++j) {
                    const zc m = zsub(DZ(i, j), zmul(zmul(ctau, v[i]), p[j]));
                    dot = zadd(dot, zmul(m, v[j]));
                }
                w2[i] = dot;
            }
        }
        __syncthreads();
        // --- second halves, element-wise, all threads: thread = row i (contiguous in memory), ty strides the columns
        {
            const int ty = tid >> 7, i = tid & 127;
            if (i < L) {
                const zc cv = zmul(ctau, v[i]);
                for (int64_t j0 = c + 1 + ty; j0 < r0; j0 += 24) {
                    zc e[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if (j0 + 3 * u < r0) e[u] = BC_Z(r0 + i, j0 + 3 * u);
#pragma unroll
                    for (int u = 0; u < 8; ++u)
                        if (j0 + 3 * u < r0) BC_Z(r0 + i, j0 + 3 * u) = zsub(e[u], zmul(cv, dA[j0 + 3 * u - (c + 1)]));
                }
                for (int j = ty; j <= i; j += 3) {
                    const zc m = zsub(TD[toff(j) + i - j], zmul(zmul(ctau, v[i]), p[j]));
                    zc r = zsub(m, zmul(zmul(tau, w2[i]), zconj(v[j])));
                    if (i == j) r.im = 0.0;              // a Hermitian diagonal is real
                    BC_Z(r0 + i, r0 + j) = r;
                }
            }
        }
#undef DZ
        return;
    }
    // With 384 threads (persistent kernel) three groups of 128 run the disjoint blocks (i), (iii), (ii) side
    // by side ((ii) synchronises on a named barrier of its own); with fewer threads they run one after
    // the other.  Same arithmetic either way.
    const bool par = nt >= 384;
    const int grp = par ? (tid >> 7) : 0, t0 = par ? (tid & 127) : tid, st_ = par ? 128 : nt;
    auto sync_ii = [&]() {
        if (par)
            asm volatile("bar.sync 1, 128;" ::: "memory");
        else
            __syncthreads();
    };
    if (!par || grp == 0) {
        // --- (i) A <- H^H A = A - conj(tau) v (v^H A)
        for (int64_t j = c + 1 + t0; j < r0; j += st_) {
            zc dot = {0.0, 0.0};
            for (int i = 0; i < L; ++i) dot = zadd(dot, zmul(zconj(v[i]), BC_Z(r0 + i, j)));
            for (int i = 0; i < L; ++i) BC_Z(r0 + i, j) = zsub(BC_Z(r0 + i, j), zmul(zmul(ctau, v[i]), dot));
        }
    }
    if (!par || grp == 2) {
        // --- (ii) D <- H^H D H: p = v^H D;  M = D - conj(tau) v p;  w2 = M v;  D' = M - tau w2 v^H (lower part)
        for (int j = t0; j < L; j += st_) {
            zc dot = {0.0, 0.0};
            for (int i = 0; i < L; ++i)
                dot = zadd(dot, zmul(zconj(v[i]), (i >= j) ? BC_Z(r0 + i, r0 + j) : zconj(BC_Z(r0 + j, r0 + i))));
            p[j] = dot;
        }
        sync_ii();
        for (int i = t0; i < L; i += st_) {
            zc dot = {0.0, 0.0};
            for (int j = 0; j < L; ++j) {
                const zc dij = (i >= j) ? BC_Z(r0 + i, r0 + j) : zconj(BC_Z(r0 + j, r0 + i));
                const zc m = zsub(dij, zmul(zmul(ctau, v[i]), p[j]));
                dot = zadd(dot, zmul(m, v[j]));
            }
            w2[i] = dot;
        }
        sync_ii();
        for (int j = t0; j < L; j += st_)
            for (int i = j; i < L; ++i) {
                const zc m = zsub(BC_Z(r0 + i, r0 + j), zmul(zmul(ctau, v[i]), p[j]));
                zc r = zsub(m, zmul(zmul(tau, w2[i]), zconj(v[j])));
                if (i == j) r.im = 0.0;              // a Hermitian diagonal is real
                BC_Z(r0 + i, r0 + j) = r;
            }
    }
    if (!par || grp == 1) {
        // --- (iii) E <- E H = E - tau (E v) v^H
        int64_t r2 = r1 + NBW;
        if (r2 > N - 1) r2 = N - 1;
        for (int64_t i = r1 + 1 + t0; i <= r2; i += st_) {
            if (need_head && i == r2) {          // the corner is the head element of step (s-1, k+2): wait for its beta
                uint32_t h;
                do {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(h) : "l"(head_prev) : "memory");
                } while (h < need_head);
            }
            zc dot = {0.0, 0.0};
            for (int l = 0; l < L; ++l) dot = zadd(dot, zmul(BC_Z(i, r0 + l), v[l]));
            for (int l = 0; l < L; ++l) BC_Z(i, r0 + l) = zsub(BC_Z(i, r0 + l), zmul(zmul(tau, dot), zconj(v[l])));
        }
    }
#undef BC_Z
}

template <int NBW>
__global__ void __launch_bounds__(128) bc_wavefront_kernel_z(int64_t N, int64_t t, int64_t s_hi, zc *__restrict__ ab,
                                                             zc *__restrict__ hh_v, zc *__restrict__ hh_tau)
{
    constexpr int LG = (NBW == 32) ? 5 : (NBW == 64) ? 6 : 7;
    __shared__ zc v[NBW], p[NBW], w2[NBW], zsc[2];
    __shared__ double dsc[1];
    const int64_t s = s_hi - blockIdx.x;
    if (s < 0) return;
    const int64_t k = t - 3 * s;
    const int64_t K = (N - 1 - s + NBW - 1) >> LG;
    if (k < 0 || k >= K) return;
    bc_step_global_z<NBW>(N, s, k, ab, hh_v, hh_tau, v, p, w2, zsc, dsc);
}

// persistent complex version (nbw = 128): same flags and 2-step lag as bc_persistent_kernel; block (ii) in
// shared memory, block (i) streamed through it (TD in bc_step_global_z)
template <int NBW>
__global__ void __launch_bounds__(384) bc_persistent_kernel_z(int64_t N, zc *__restrict__ ab, zc *__restrict__ hh_v,
                                                              zc *__restrict__ hh_tau, uint32_t *__restrict__ prog)
{
    constexpr int LG = (NBW == 32) ? 5 : (NBW == 64) ? 6 : 7;
    extern __shared__ __align__(16) unsigned char zsm_td[];      // packed triangle of the diagonal block + NBW dots
    zc *TD = reinterpret_cast<zc *>(zsm_td);
    __shared__ zc v[NBW], p[NBW], w2[NBW], zsc[2];
    __shared__ double dsc[1];
    const int tid = threadIdx.x;
    uint32_t *done = prog, *head = prog + N;
    for (int64_t s = blockIdx.x; s <= N - 2; s += gridDim.x) {
        const int64_t K = (N - 1 - s + NBW - 1) >> LG;
        const int64_t Kprev = (N - s + NBW - 1) >> LG;
        uint32_t known = 0;
        for (int64_t k = 0; k < K; ++k) {
            uint32_t need_head = 0;
            if (s > 0) {
                const uint32_t need = (uint32_t)((k + 2 < Kprev) ? k + 2 : Kprev);
                if (tid == 0) {
                    while (known < need) {
                        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(known) : "l"(done + s - 1) : "memory");
                    }
                }
                __syncthreads();
                if (k + 2 < Kprev) need_head = (uint32_t)(k + 3);
            }
            bc_step_global_z<NBW>(N, s, k, ab, hh_v, hh_tau, v, p, w2, zsc, dsc, head + s, head + s - 1, need_head, TD);
            // the CTA barrier orders every thread's stores before thread 0's release (the pattern grid-wide
            // barriers are built from): one fence, not one per thread
            __syncthreads();
            if (tid == 0) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(done + s), "r"((uint32_t)(k + 1)) : "memory");
        }
    }
}

// ---- complex step with its blocks staged in shared memory (nbw <= 64) ----------------------------------
// Two tiles: TA = block (i), nA columns x L rows (column stride NBW+1 elements); TB = blocks (ii)+(iii),
// L columns x nR rows (column stride 2 NBW + 1): 198 KB at nbw = 64.  Arithmetic as bc_step_global_z.
template <int NBW>
__device__ __forceinline__ bool bc_step_smem_z(const int64_t N, const int64_t s, const int64_t k, zc *__restrict__ ab,
                                               zc *__restrict__ hh_v, zc *__restrict__ hh_tau, zc *TA, zc *TB, zc *v, zc *p,
                                               zc *w2, zc *zsc, double *dsc, uint32_t *head_mine,
                                               const uint32_t *head_prev, const uint32_t need_head, const bool e_in)
{
    // e_in / return value: block (iii) handed from step to step in shared memory, as in bc_step_smem
    constexpr int LG = (NBW == 32) ? 5 : 6;
    constexpr int64_t ldab = 2 * NBW + 1;
    constexpr int LDA = NBW + 1, LDB = 2 * NBW + 1;
    const int tid = threadIdx.x, nt = blockDim.x;
    const int64_t r0 = s + 1 + (k << LG);
    int64_t r1 = s + ((k + 1) << LG);
    if (r1 > N - 1) r1 = N - 1;
    const int L = (int)(r1 - r0 + 1);
    const int64_t c = (k == 0) ? s : r0 - NBW;
    const int64_t g = hh_off(N, NBW, s) + k;
    zc *vout = hh_v + g * NBW;
    if (k > 0 && L == 1) {
        for (int i = tid; i < NBW; i += nt) vout[i] = {(i == 0) ? 1.0 : 0.0, 0.0};
        if (tid == 0) {
            hh_tau[g] = {0.0, 0.0};
            asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(head_mine), "r"((uint32_t)(k + 1)) : "memory");
        }
        return false;
    }
    int64_t r2 = r1 + NBW;
    if (r2 > N - 1) r2 = N - 1;
    const int nA = (int)(r0 - c - 1), nR = (int)(r2 - r0 + 1);
    // element (r0 + row, col j) of the band: ab[(r0 + row - j) + j * ldab]
    const bool keep = (nR - L >= 2);              // the next step (L' = nR - L rows) takes block (iii) from TB
    const int warp = tid >> 5, lane = tid & 31, nwarp = nt >> 5;
    int qs = 0;
    if (e_in) {
        // previous step: L = NBW; its block (iii) = TB rows NBW .. NBW+L-1: column 0 is x, columns 1.. block (i)
        if (tid < L) p[tid] = TB[NBW + tid];
        for (int q = warp; q < NBW - 1; q += nwarp)
            for (int row = lane; row < L; row += 32) TA[q * LDA + row] = TB[(q + 1) * LDB + NBW + row];
        __syncthreads();
        qs = nA;
    }
    for (int q = qs + warp; q < nA + L; q += nwarp) {     // a warp per column, lanes along its band segment
        const int64_t j = c + 1 + q;
        const zc *src = ab + (r0 - j) + j * ldab;
        zc *dst = (q < nA) ? TA + q * LDA : TB + (q - nA) * LDB;
        const int lo = (q < nA) ? 0 : q - nA, hi = (q < nA) ? L : nR;
        for (int row = lo + lane; row < hi; row += 32) cp_async16(smem_u32(dst + row), src + row, 16u);
    }
    cp_async_commit();
    if (!e_in && tid < L) p[tid] = ab[(r0 + tid - c) + c * ldab];
    cp_async_wait_all();
    __syncthreads();
    if (tid == 0) {
        const double ar = p[0].re, ai = p[0].im;
        double ss = 0.0;
#pragma unroll 8
        for (int i = 1; i < L; ++i) ss = __dadd_rn(ss, __dadd_rn(__dmul_rn(p[i].re, p[i].re), __dmul_rn(p[i].im, p[i].im)));
        if (ss == 0.0 && ai == 0.0) {
            zsc[0] = {0.0, 0.0};
            zsc[1] = {0.0, 0.0};
            dsc[0] = ar;
        } else {
            const double nrm = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(ar, ar), __dmul_rn(ai, ai)), ss));
            const double b = (ar >= 0.0) ? -nrm : nrm;
            zsc[0] = {__ddiv_rn(__dsub_rn(b, ar), b), __ddiv_rn(-ai, b)};
            zsc[1] = zrecip({__dsub_rn(ar, b), ai});
            dsc[0] = b;
        }
    }
    __syncthreads();
    const zc tau = zsc[0], ctau = zconj(zsc[0]);
    const bool ident = (tau.re == 0.0 && tau.im == 0.0);
    for (int i = tid; i < NBW; i += nt) {
        zc vi = {0.0, 0.0};
        if (i == 0) vi = {1.0, 0.0};
        else if (i < L && !ident) vi = zmul(p[i], zsc[1]);
        v[i] = vi;
        vout[i] = vi;
    }
    if (tid < L) ab[(r0 + tid - c) + c * ldab] = {(tid == 0) ? dsc[0] : 0.0, 0.0};
    if (tid == 0) {
        hh_tau[g] = tau;
        asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(head_mine), "r"((uint32_t)(k + 1)) : "memory");
    }
    __syncthreads();
    if (ident && !e_in) return false;
#define ZA(rl, q) TA[(q) * LDA + (rl)]
#define ZB(rl, q) TB[(q) * LDB + (rl)]
    const int grp = ident ? 3 : (tid >> 6), t64 = tid & 63;
    if (grp == 3) {
        // identity step holding the previous step's block (iii): re-fetch the corner once step (s-1, k+2)
        // has written its beta there, as group 1 does (see bc_step_smem)
        if (need_head && tid == 0 && nR > L) {
            uint32_t h;
            do {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(h) : "l"(head_prev) : "memory");
            } while (h < need_head);
            const int64_t jc = r0 + L - 1;
            const double2 cv = __ldcg(reinterpret_cast<const double2 *>(&ab[(r0 + nR - 1 - jc) + jc * ldab]));
            ZB(nR - 1, L - 1) = {cv.x, cv.y};
        }
    } else if (grp == 0) {
        // --- (i) A <- H^H A = A - conj(tau) v (v^H A)
        for (int q = t64; q < nA; q += 64) {
            zc dot = {0.0, 0.0};
#pragma unroll 4
            for (int i = 0; i < L; ++i) dot = zadd(dot, zmul(zconj(v[i]), ZA(i, q)));
#pragma unroll 4
            for (int i = 0; i < L; ++i) ZA(i, q) = zsub(ZA(i, q), zmul(zmul(ctau, v[i]), dot));
        }
    } else if (grp == 1) {
        // --- (iii) E <- E H = E - tau (E v) v^H
        for (int rl = L + t64; rl < nR; rl += 64) {
            if (need_head && rl == nR - 1) {
                uint32_t h;
                do {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(h) : "l"(head_prev) : "memory");
                } while (h < need_head);
                const int64_t jc = r0 + L - 1;
                const double2 cv = __ldcg(reinterpret_cast<const double2 *>(&ab[(r0 + rl - jc) + jc * ldab]));
                ZB(rl, L - 1) = {cv.x, cv.y};
            }
            zc dot = {0.0, 0.0};
#pragma unroll 4
            for (int l = 0; l < L; ++l) dot = zadd(dot, zmul(ZB(rl, l), v[l]));
#pragma unroll 4
            for (int l = 0; l < L; ++l) ZB(rl, l) = zsub(ZB(rl, l), zmul(zmul(tau, dot), zconj(v[l])));
        }
    } else if (grp == 2) {
        // --- (ii) D(i, j) = ZB(i, j) (i >= j) or conj(ZB(j, i))
        for (int j = t64; j < L; j += 64) {
            zc dot = {0.0, 0.0};
#pragma unroll 4
            for (int i = 0; i < L; ++i) dot = zadd(dot, zmul(zconj(v[i]), (i >= j) ? ZB(i, j) : zconj(ZB(j, i))));
            p[j] = dot;
        }
        asm volatile("bar.sync 1, 64;" ::: "memory");
        for (int i = t64; i < L; i += 64) {
            zc dot = {0.0, 0.0};
#pragma unroll 4
            for (int j = 0; j < L; ++j) {
                const zc dij = (i >= j) ? ZB(i, j) : zconj(ZB(j, i));
                const zc m = zsub(dij, zmul(zmul(ctau, v[i]), p[j]));
                dot = zadd(dot, zmul(m, v[j]));
            }
            w2[i] = dot;
        }
        asm volatile("bar.sync 1, 64;" ::: "memory");
        for (int j = t64; j < L; j += 64)
            for (int i = j; i < L; ++i) {
                const zc m = zsub(ZB(i, j), zmul(zmul(ctau, v[i]), p[j]));
                zc r = zsub(m, zmul(zmul(tau, w2[i]), zconj(v[j])));
                if (i == j) r.im = 0.0;
                ZB(i, j) = r;
            }
    }
    __syncthreads();
#undef ZA
#undef ZB
    // two columns at a time through registers (both columns' shared-memory loads in flight together, as in
    // the real step)
    for (int q = warp; q < nA + L; q += 2 * nwarp) {
        zc t0[4], t1[4];
        const int q1 = q + nwarp;
        const bool two = q1 < nA + L;
        const zc *s0 = (q < nA) ? TA + q * LDA : TB + (q - nA) * LDB;
        const zc *s1 = (q1 < nA) ? TA + q1 * LDA : TB + (q1 - nA) * LDB;
        const int lo0 = (q < nA) ? 0 : q - nA, hi0 = (q < nA) ? L : (keep ? L : nR);
        const int lo1 = (q1 < nA) ? 0 : q1 - nA, hi1 = two ? ((q1 < nA) ? L : (keep ? L : nR)) : 0;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int ra = lo0 + lane + 32 * u, rb = lo1 + lane + 32 * u;
            if (ra < hi0) t0[u] = s0[ra];
            if (rb < hi1) t1[u] = s1[rb];
        }
        const int64_t j0 = c + 1 + q, j1 = c + 1 + q1;
        zc *d0 = ab + (r0 - j0) + j0 * ldab, *d1 = ab + (r0 - j1) + j1 * ldab;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int ra = lo0 + lane + 32 * u, rb = lo1 + lane + 32 * u;
            if (ra < hi0) d0[ra] = t0[u];
            if (rb < hi1) d1[rb] = t1[u];
        }
    }
    return keep;
}

template <int NBW>
__global__ void __launch_bounds__(256) bc_persistent_smem_kernel_z(int64_t N, zc *__restrict__ ab, zc *__restrict__ hh_v,
                                                                   zc *__restrict__ hh_tau, uint32_t *__restrict__ prog)
{
    constexpr int LG = (NBW == 32) ? 5 : 6;
    extern __shared__ __align__(16) unsigned char zsm[];
    zc *TA = reinterpret_cast<zc *>(zsm);
    zc *TB = TA + (NBW - 1) * (NBW + 1);
    __shared__ zc v[NBW], p[NBW], w2[NBW], zsc[2];
    __shared__ double dsc[1];
    const int tid = threadIdx.x;
    uint32_t *done = prog, *head = prog + N;
    for (int64_t s = blockIdx.x; s <= N - 2; s += gridDim.x) {
        const int64_t K = (N - 1 - s + NBW - 1) >> LG;
        const int64_t Kprev = (N - s + NBW - 1) >> LG;
        uint32_t known = 0;
        bool e_in = false;
        for (int64_t k = 0; k < K; ++k) {
            uint32_t need_head = 0;
            if (s > 0) {
                const uint32_t need = (uint32_t)((k + 2 < Kprev) ? k + 2 : Kprev);
                if (tid == 0) {
                    while (known < need) {
                        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(known) : "l"(done + s - 1) : "memory");
                    }
                }
                __syncthreads();
                if (k + 2 < Kprev) need_head = (uint32_t)(k + 3);
            }
            e_in = bc_step_smem_z<NBW>(N, s, k, ab, hh_v, hh_tau, TA, TB, v, p, w2, zsc, dsc, head + s, head + s - 1, need_head, e_in);
            // the CTA barrier orders every thread's stores before thread 0's release (the pattern grid-wide
            // barriers are built from): one fence, not one per thread
            __syncthreads();
            if (tid == 0) asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(done + s), "r"((uint32_t)(k + 1)) : "memory");
        }
    }
}

template <int NBW>
__global__ void bc_extract_kernel_z(int64_t N, const zc *__restrict__ ab, double *__restrict__ d, double *__restrict__ e)
{
    constexpr int64_t ldab = 2 * NBW + 1;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) d[i] = ab[i * ldab].re;
    if (i + 1 < N) e[i] = ab[1 + i * ldab].re;
}

// d[i] = T[i][i], e[i] = T[i+1][i]
template <int NBW>
__global__ void bc_extract_kernel(int64_t N, const double *__restrict__ ab, double *__restrict__ d, double *__restrict__ e)
{
    constexpr int64_t ldab = 2 * NBW + 1;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) d[i] = ab[i * ldab];
    if (i + 1 < N) e[i] = ab[1 + i * ldab];
}

// The persistent kernels wait on flags written by other CTAs of the same grid, so every CTA of the grid
// must be resident at once: a cooperative launch (no grid.sync is used) makes the driver guarantee that,
// or fail, instead of leaving it to how busy the device happens to be.
template <class K, class T>
cudaError_t bc_launch_persistent(K kern, int64_t grid, int threads, size_t smem, cudaStream_t st, int64_t N, T *ab, T *hh_v,
                                 T *hh_tau, uint32_t *prog)
{
    void *args[] = {(void *)&N, (void *)&ab, (void *)&hh_v, (void *)&hh_tau, (void *)&prog};
    return cudaLaunchCooperativeKernel((const void *)kern, dim3((unsigned)grid), dim3((unsigned)threads), args, smem, st);
}

// host: prog == nullptr (or nbw = 128): all wavefronts t = 3s + k, in order, on one stream;
// otherwise the persistent kernel (prog: 2 N zeroed counters).  *launches = kernels launched.
template <int NBW>
cudaError_t launch_bulge_chase(int64_t N, double *ab, double *hh_v, double *hh_tau, double *d, double *e,
                               cudaStream_t st, int64_t *launches, uint32_t *prog = nullptr, int nsm = 0)
{
    constexpr int LG = (NBW == 32) ? 5 : (NBW == 64) ? 6 : 7;
    int64_t nl = 0;
    constexpr int smem_bytes = (2 * NBW - 1) * (2 * NBW + 1) * 8;
    if (NBW <= 64) {
        cudaError_t e0 = set_max_smem((const void *)bc_wavefront_smem_kernel<(NBW <= 64 ? NBW : 64)>, smem_bytes);
        if (e0 != cudaSuccess) return e0;
    }
    if (NBW > 64 && prog && nsm > 0 && N >= 2) {
        const int64_t grid = (N - 1 < nsm) ? N - 1 : nsm;
        // triangle of block (ii) + NBW dot products + the tile of block (i)
        constexpr int tbytes = (NBW * (NBW + 1) / 2 + NBW + (NBW - 1) * (NBW + 1)) * 8;
        cudaError_t e0 = set_max_smem((const void *)bc_persistent_global_kernel<NBW>, tbytes);
        if (e0 != cudaSuccess) return e0;
        cudaError_t e1 = bc_launch_persistent(bc_persistent_global_kernel<NBW>, grid, 384, tbytes, st, N, ab, hh_v, hh_tau, prog);
        ++nl;
        if (e1 != cudaSuccess) return e1;
    } else if (NBW <= 64 && prog && nsm > 0 && N >= 2) {
        auto pk = bc_persistent_kernel<(NBW <= 64 ? NBW : 64)>;
        cudaError_t e0 = set_max_smem((const void *)pk, smem_bytes);
        if (e0 != cudaSuccess) return e0;
        // one CTA per SM (its tile takes more than half of an SM's shared memory): all CTAs are resident,
        // which the flag waits between sweeps rely on
        const int64_t grid = (N - 1 < nsm) ? N - 1 : nsm;
        cudaError_t e1 = bc_launch_persistent(pk, grid, 256, smem_bytes, st, N, ab, hh_v, hh_tau, prog);
        ++nl;
        if (e1 != cudaSuccess) return e1;
    } else if (N >= 2) {
        const int64_t Kmax = (N - 2 + NBW) >> LG;                  // K(0)
        // last wavefront: max over s of 3s + K(s) - 1; K(s) >= 1 for s <= N-2, so s = N-2 gives 3(N-2)
        int64_t tmax = 0;
        for (int64_t s = (N > 2 + Kmax) ? N - 2 - Kmax : 0; s <= N - 2; ++s) {
            const int64_t K = (N - 1 - s + NBW - 1) >> LG;
            if (3 * s + K - 1 > tmax) tmax = 3 * s + K - 1;
        }
        if (Kmax - 1 > tmax) tmax = Kmax - 1;
        for (int64_t t = 0; t <= tmax; ++t) {
            int64_t s_hi = t / 3;
            if (s_hi > N - 2) s_hi = N - 2;
            int64_t s_lo = (t - Kmax + 1 + 2) / 3;                 // k = t - 3s <= Kmax - 1
            if (t - Kmax + 1 <= 0) s_lo = 0;
            if (s_lo > s_hi) continue;
            if (NBW <= 64)
                bc_wavefront_smem_kernel<(NBW <= 64 ? NBW : 64)>
                    <<<(unsigned)(s_hi - s_lo + 1), 256, smem_bytes, st>>>(N, t, s_hi, ab, hh_v, hh_tau);
            else
                bc_wavefront_kernel<NBW><<<(unsigned)(s_hi - s_lo + 1), 128, 0, st>>>(N, t, s_hi, ab, hh_v, hh_tau);
            ++nl;
        }
        cudaError_t e1 = cudaGetLastError();
        if (e1 != cudaSuccess) return e1;
    }
    if (N >= 1) {
        bc_extract_kernel<NBW><<<(unsigned)((N + 255) / 256), 256, 0, st>>>(N, ab, d, e);
        ++nl;
    }
    if (launches) *launches = nl;
    return cudaGetLastError();
}

// complex: the same wavefronts, global-memory step
template <int NBW>
cudaError_t launch_bulge_chase_z(int64_t N, zc *ab, zc *hh_v, zc *hh_tau, double *d, double *e, cudaStream_t st,
                                 int64_t *launches, uint32_t *prog = nullptr, int nsm = 0)
{
    constexpr int LG = (NBW == 32) ? 5 : (NBW == 64) ? 6 : 7;
    int64_t nl = 0;
    if (prog && nsm > 0 && N >= 2) {
        // one CTA per SM: resident by construction (the flag waits between sweeps rely on it)
        const int64_t grid = (N - 1 < nsm) ? N - 1 : nsm;
        cudaError_t e1 = cudaSuccess;
        if (NBW <= 64) {
            constexpr int NB = (NBW <= 64) ? NBW : 64;
            constexpr int zbytes = ((NB - 1) * (NB + 1) + NB * (2 * NB + 1)) * 16;
            auto zk = bc_persistent_smem_kernel_z<NB>;
            cudaError_t e0 = set_max_smem((const void *)zk, zbytes);
            if (e0 != cudaSuccess) return e0;
            e1 = bc_launch_persistent(zk, grid, 256, zbytes, st, N, ab, hh_v, hh_tau, prog);
        } else {
            // triangle of block (ii) + NBW dot products + two 16-row chunk buffers of block (i)
            constexpr int tbytes = (NBW * (NBW + 1) / 2 + NBW + 2 * (NBW - 1) * 17) * 16;
            cudaError_t e0 = set_max_smem((const void *)bc_persistent_kernel_z<NBW>, tbytes);
            if (e0 != cudaSuccess) return e0;
            e1 = bc_launch_persistent(bc_persistent_kernel_z<NBW>, grid, 384, tbytes, st, N, ab, hh_v, hh_tau, prog);
        }
        ++nl;
        if (e1 != cudaSuccess) return e1;
    } else if (N >= 2) {
        const int64_t Kmax = (N - 2 + NBW) >> LG;
        const int64_t tmax = (3 * (N - 2) > Kmax - 1) ? 3 * (N - 2) : Kmax - 1;
        for (int64_t t = 0; t <= tmax; ++t) {
            int64_t s_hi = t / 3;
            if (s_hi > N - 2) s_hi = N - 2;
            int64_t s_lo = (t - Kmax + 1 + 2) / 3;
            if (t - Kmax + 1 <= 0) s_lo = 0;
            if (s_lo > s_hi) continue;
            bc_wavefront_kernel_z<NBW><<<(unsigned)(s_hi - s_lo + 1), 128, 0, st>>>(N, t, s_hi, ab, hh_v, hh_tau);
            ++nl;
        }
        cudaError_t e1 = cudaGetLastError();
        if (e1 != cudaSuccess) return e1;
    }
    if (N >= 1) {
        bc_extract_kernel_z<NBW><<<(unsigned)((N + 255) / 256), 256, 0, st>>>(N, ab, d, e);
        ++nl;
    }
    if (launches) *launches = nl;
    return cudaGetLastError();
}

}  // namespace elpa2bt
