// bt_f32.cuh -- SURVEY.md 8(f) NEXT-4: the tridiagonal -> band back-transformation (Eq. 6d PAPER.md:91,
// Eq. 8) in FP32, real and complex (R16), sm_100a.
//
// There is no FP32 tensor-core type on sm_100a (TF32 drops 13 mantissa bits), so this is the north
// star's "reflector path" on the FP32 FMA pipe (148 SMs x 128 FFMA/clk), one reflector at a time
// exactly as Eq. 8 states it -- no aggregation, every useful flop is one FFMA:
//
//  * a lane owns ONE column of q; its window of W = nbw + 8 rows sits in registers (complex: planar);
//    a warp owns a strip of 32 columns and walks the chains k = 0 .. K0-1 (chain-major order, R5);
//  * a block = the 8 consecutive reflectors of a chain with first rows 8b+7 .. 8b (the block structure
//    of bt_wy.cuh); reflector i acts on window offsets 7-i .. 7-i+nbw-1, all register indices are
//    compile-time constants.  v and tau come from shared memory by broadcast LDS.128 (one address
//    per warp), staged per CTA by 16-byte cp.async into an 8-stage ring (full / empty mbarriers, the
//    warps take turns at staging as in bt_wy.cuh);
//  * the window moves up 8 rows per block: the update of the block's last reflector
//    writes its result 8 registers further on, the 8 rows on top retire to global memory (32 contiguous
//    bytes per column and lane: one full sector), the next 8 rows are loaded one block ahead.
// Model work 4 L flops per reflector and column (16 L complex) = 2 L FFMAs (8 L): the FFMA count is
// the model's, the ceiling is set by the LDS : FFMA issue ratio (1 : 4 real, 1 : 8 complex).
#pragma once
#include "bt_common.cuh"
#include "bt_wy.cuh"        // block enumeration (wy_bhi, wy_nchains, wy_slot), cp_async_mbar_arrive_noinc_wy

namespace elpa2bt {

template <bool CPLX_, int NBW_>
struct F32Cfg {
    static constexpr bool CPLX = CPLX_;
    static constexpr int NBW = NBW_;
    static constexpr int EW = CPLX ? 2 : 1;           // floats per element
    static constexpr int NB8 = NBW / 8;
    static constexpr int W = NBW + 8;                 // window rows
    static constexpr int NW = 8;                      // warps per CTA
    static constexpr int NS = 8, LGNS = 3, LAG = 4;   // ring
    static constexpr int V_FLOATS = 8 * NBW * EW;     // V[i][r] (interleaved for complex)
    static constexpr int STAGE_FLOATS = V_FLOATS + 16;// + tau[8] (re, im)
    // per-warp ring of incoming 8-row tiles of q: [16-byte piece][lane][4 floats], filled by the lane's own cp.async
    static constexpr int NSQ = 4, DQ = 3;             // stages, tiles fetched ahead
    static constexpr int QTILE = 8 * 32 * EW;         // floats per tile
    static constexpr int OFF_Q = NS * STAGE_FLOATS * 4;
    static constexpr int OFF_BAR = OFF_Q + NW * NSQ * QTILE * 4;
    static constexpr int SMEM_BYTES = OFF_BAR + 2 * NS * 8;
    static_assert(NBW % 32 == 0, "nbw");
};

struct F32Args {
    int64_t N, nev, ldq;
    const float *hh_v;     // G * nbw elements
    const float *hh_tau;   // G elements
    float *q;
    int align16;           // q base and ldq * element size are 16-byte aligned
};

__device__ __forceinline__ void cp_async4(uint32_t dst, const void *src, uint32_t src_bytes)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}

// ---- staging one block (whole warp): 8 reflectors of nbw elements + their tau ---------------------------
template <class C>
__device__ __forceinline__ void f32_stage(const F32Args &a, float *stage, uint32_t bar_full, int64_t k, int64_t b,
                                          int64_t FN1, int lane)
{
    constexpr int NBW = C::NBW, EW = C::EW;
    constexpr int CPR = NBW * EW / 4;                 // 16-byte chunks per reflector
    const int64_t myslot = wy_slot<NBW>(a.N, FN1, k, b, lane & 7);
#pragma unroll
    for (int t = 0; t < 8 * CPR / 32; ++t) {
        const int c = t * 32 + lane, i = c / CPR, j = c % CPR;
        const int64_t sl = __shfl_sync(0xffffffffu, myslot, i);
        const float *src = a.hh_v + (sl >= 0 ? sl : 0) * (NBW * EW) + 4 * j;
        cp_async16(smem_u32(stage + i * (NBW * EW) + 4 * j), src, sl >= 0 ? 16u : 0u);
    }
    if (lane < 8) {
        const float *src = a.hh_tau + (myslot >= 0 ? myslot : 0) * EW;
        if (EW == 2)
            cp_async8(smem_u32(stage + C::V_FLOATS + 2 * lane), src, myslot >= 0 ? 8u : 0u);
        else
            cp_async4(smem_u32(stage + C::V_FLOATS + 2 * lane), src, myslot >= 0 ? 4u : 0u);
    }
    cp_async_mbar_arrive_noinc_wy(bar_full);
}

// ---- 8 rows of this lane's column (rows row0 .. row0+7, row0 a multiple of 8) on their way in ---------------------
// f32_fetch8: the lane's own cp.async copies into its slots of the warp's tile (zero fill beyond N and for
// absent columns / blocks); f32_take8: the same lane reads them back once its copy group has completed.
template <bool CPLX>
__device__ __forceinline__ void f32_fetch8(const F32Args &a, const float *colp, bool ok, int64_t row0, float *tile, int lane)
{
    constexpr int EW = CPLX ? 2 : 1, NP = 2 * EW;     // 16-byte pieces: 4 / EW rows each
    const int64_t left = ok ? a.N - row0 : 0;         // rows present from row0 on
    if (a.align16) {
#pragma unroll
        for (int h = 0; h < NP; ++h) {
            int64_t nr = left - h * (4 / EW);
            nr = nr < 0 ? 0 : (nr > 4 / EW ? 4 / EW : nr);
            cp_async16(smem_u32(tile + (h * 32 + lane) * 4), nr ? colp + (row0 * EW + 4 * h) : a.q, (uint32_t)(nr * 4 * EW));
        }
    } else {
#pragma unroll
        for (int e = 0; e < 8 * EW; ++e) {
            const bool in = (e / EW) < left;
            cp_async4(smem_u32(tile + ((e >> 2) * 32 + lane) * 4 + (e & 3)), in ? colp + (row0 * EW + e) : a.q, in ? 4u : 0u);
        }
    }
}
template <bool CPLX>
__device__ __forceinline__ void f32_take8(const float *tile, int lane, float *r, float *im)
{
    if (CPLX) {
#pragma unroll
        for (int h = 0; h < 4; ++h) {
            const float4 v = *reinterpret_cast<const float4 *>(tile + (h * 32 + lane) * 4);
            r[2 * h] = v.x, im[2 * h] = v.y, r[2 * h + 1] = v.z, im[2 * h + 1] = v.w;
        }
    } else {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const float4 v = *reinterpret_cast<const float4 *>(tile + (h * 32 + lane) * 4);
            r[4 * h] = v.x, r[4 * h + 1] = v.y, r[4 * h + 2] = v.z, r[4 * h + 3] = v.w;
        }
    }
}

template <bool CPLX>
__device__ __forceinline__ void f32_store8(const F32Args &a, float *colp, bool colok, int64_t row0, const float *r,
                                           const float *im)
{
    if (!colok || row0 >= a.N) return;
    if (a.align16 && row0 + 8 <= a.N) {
        if (CPLX) {
#pragma unroll
            for (int h = 0; h < 4; ++h)
                *reinterpret_cast<float4 *>(colp + 2 * row0 + 4 * h) = make_float4(r[2 * h], im[2 * h], r[2 * h + 1], im[2 * h + 1]);
        } else {
#pragma unroll
            for (int h = 0; h < 2; ++h)
                *reinterpret_cast<float4 *>(colp + row0 + 4 * h) = make_float4(r[4 * h], r[4 * h + 1], r[4 * h + 2], r[4 * h + 3]);
        }
        return;
    }
#pragma unroll
    for (int e = 0; e < 8; ++e)
        if (row0 + e < a.N) {
            if (CPLX) {
                colp[2 * (row0 + e)] = r[e];
                colp[2 * (row0 + e) + 1] = im[e];
            } else {
                colp[row0 + e] = r[e];
            }
        }
}

// ---- reading a reflector from shared memory ----------------------------------------------------------------
// body(j, v4) for the NL broadcast LDS.128 of a reflector, ascending (dot product) or descending (update).
// CH = 0: plain loads; ptxas keeps the reflector in registers between the two passes and hoists loads as it
// likes -- right for narrow windows.  CH > 0 (wide windows, where that costs spills): the loads go in
// chunks of CH, chunk c+1 issued before the arithmetic of chunk c, and a __syncwarp() between chunks keeps
// later loads from being hoisted above it (it orders shared-memory accesses): at most 2 CH float4 are live.
template <int NL, int CH, bool DESC, class F>
__device__ __forceinline__ void f32_for_v(const float *v, F &&body)
{
    if constexpr (CH == 0) {
#pragma unroll
        for (int t = 0; t < NL; ++t) {
            const int j = DESC ? NL - 1 - t : t;
            body(j, *reinterpret_cast<const float4 *>(v + 4 * j));
        }
    } else {
        constexpr int NC = NL / CH;
        static_assert(NL % CH == 0, "chunking");
        float4 buf[2][CH];
#pragma unroll
        for (int t = 0; t < CH; ++t) buf[0][t] = *reinterpret_cast<const float4 *>(v + 4 * (DESC ? NL - 1 - t : t));
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            __syncwarp();
            if (c + 1 < NC) {
#pragma unroll
                for (int t = 0; t < CH; ++t) {
                    const int j = DESC ? NL - 1 - ((c + 1) * CH + t) : (c + 1) * CH + t;
                    buf[(c + 1) & 1][t] = *reinterpret_cast<const float4 *>(v + 4 * j);
                }
            }
#pragma unroll
            for (int t = 0; t < CH; ++t) body(DESC ? NL - 1 - (c * CH + t) : c * CH + t, buf[c & 1][t]);
        }
    }
}

// ---- one reflector on the register window --------------------------------------------------------------
// x[OFF + r] -= tau (v^H x) v[r], r < nbw.  SHIFT = 8 for the block's last reflector (OFF = 0): the result
// lands 8 registers further on (the window moves up by 8 rows), written from the top down so that no
// input is overwritten before it is read.
template <int NBW, int OFF, int SHIFT>
__device__ __forceinline__ void f32_apply_real(float *x, const float *v, const float tau)
{
    constexpr int CH = (NBW > 64) ? 8 : 0;
    // eight partial sums: with at most two warps per sub-partition the dot product must bring its own
    // instruction-level parallelism (an FFMA result is ready after 4 cycles)
    float acc[8] = {0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f};
    f32_for_v<NBW / 4, CH, false>(v, [&](const int j, const float4 v4) {
        const int o = 4 * (j & 1);
        acc[o] = fmaf(v4.x, x[OFF + 4 * j], acc[o]);
        acc[o + 1] = fmaf(v4.y, x[OFF + 4 * j + 1], acc[o + 1]);
        acc[o + 2] = fmaf(v4.z, x[OFF + 4 * j + 2], acc[o + 2]);
        acc[o + 3] = fmaf(v4.w, x[OFF + 4 * j + 3], acc[o + 3]);
    });
    const float ntd = -tau * (((acc[0] + acc[4]) + (acc[1] + acc[5])) + ((acc[2] + acc[6]) + (acc[3] + acc[7])));
    f32_for_v<NBW / 4, CH, true>(v, [&](const int j, const float4 v4) {
        x[OFF + SHIFT + 4 * j + 3] = fmaf(ntd, v4.w, x[OFF + 4 * j + 3]);
        x[OFF + SHIFT + 4 * j + 2] = fmaf(ntd, v4.z, x[OFF + 4 * j + 2]);
        x[OFF + SHIFT + 4 * j + 1] = fmaf(ntd, v4.y, x[OFF + 4 * j + 1]);
        x[OFF + SHIFT + 4 * j] = fmaf(ntd, v4.x, x[OFF + 4 * j]);
    });
}

// complex: v interleaved (re, im) in shared memory, x planar in registers; tau as stored, conj(v) in the dot (R2)
template <int NBW, int OFF, int SHIFT>
__device__ __forceinline__ void f32_apply_cplx(float *xr, float *xi, const float *v, const float taur, const float taui)
{
    constexpr int CH = (NBW > 32) ? 4 : 0;
    // eight independent partial sums (see f32_apply_real)
    float dr[4] = {0.0f, 0.0f, 0.0f, 0.0f}, di[4] = {0.0f, 0.0f, 0.0f, 0.0f};
    f32_for_v<NBW / 2, CH, false>(v, [&](const int j, const float4 v4) {      // elements 2j, 2j+1
        dr[0] = fmaf(v4.x, xr[OFF + 2 * j], dr[0]);
        dr[1] = fmaf(v4.y, xi[OFF + 2 * j], dr[1]);
        di[0] = fmaf(v4.x, xi[OFF + 2 * j], di[0]);
        di[1] = fmaf(-v4.y, xr[OFF + 2 * j], di[1]);
        dr[2] = fmaf(v4.z, xr[OFF + 2 * j + 1], dr[2]);
        dr[3] = fmaf(v4.w, xi[OFF + 2 * j + 1], dr[3]);
        di[2] = fmaf(v4.z, xi[OFF + 2 * j + 1], di[2]);
        di[3] = fmaf(-v4.w, xr[OFF + 2 * j + 1], di[3]);
    });
    const float dotr = (dr[0] + dr[1]) + (dr[2] + dr[3]), doti = (di[0] + di[1]) + (di[2] + di[3]);
    const float ntr = -(taur * dotr - taui * doti), nti = -(taur * doti + taui * dotr);   // -tau * dot
    f32_for_v<NBW / 2, CH, true>(v, [&](const int j, const float4 v4) {
        // x += (ntr + i nti) (vr + i vi)
        const float r1 = fmaf(ntr, v4.z, xr[OFF + 2 * j + 1]);
        const float i1 = fmaf(ntr, v4.w, xi[OFF + 2 * j + 1]);
        xr[OFF + SHIFT + 2 * j + 1] = fmaf(-nti, v4.w, r1);
        xi[OFF + SHIFT + 2 * j + 1] = fmaf(nti, v4.z, i1);
        const float r0 = fmaf(ntr, v4.x, xr[OFF + 2 * j]);
        const float i0 = fmaf(ntr, v4.y, xi[OFF + 2 * j]);
        xr[OFF + SHIFT + 2 * j] = fmaf(-nti, v4.y, r0);
        xi[OFF + SHIFT + 2 * j] = fmaf(nti, v4.x, i0);
    });
}

// reflectors I .. END-1 of a block
template <class C, int I, int END>
__device__ __forceinline__ void f32_block_step(float *xr, float *xi, const float *V, const float *T)
{
    constexpr int NBW = C::NBW;
    if constexpr (I < END) {
        constexpr int OFF = 7 - I, SHIFT = (I == 7) ? 8 : 0;
        if constexpr (C::CPLX)
            f32_apply_cplx<NBW, OFF, SHIFT>(xr, xi, V + I * NBW * 2, T[2 * I], T[2 * I + 1]);
        else
            f32_apply_real<NBW, OFF, SHIFT>(xr, V + I * NBW, T[2 * I]);
        f32_block_step<C, I + 1, END>(xr, xi, V, T);
    }
}

// ---- a warp with one strip of 32 columns, all chains -------------------------------------------------------
template <class C>
__device__ __forceinline__ void f32_consume(const F32Args &a, unsigned char *smem, const int lane, const int member,
                                            const int nmem, const int64_t col0)
{
    constexpr int NBW = C::NBW, W = C::W, EW = C::EW, NS = C::NS, LAG = C::LAG;
    constexpr bool CPLX = C::CPLX;
    float *ring = reinterpret_cast<float *>(smem);
    const uint32_t bar_full = smem_u32(smem + C::OFF_BAR);
    const uint32_t bar_empty = bar_full + NS * 8;
    const int64_t N = a.N;
    const int64_t K0 = wy_nchains(N, NBW);
    const int64_t bhi = wy_bhi(N);
    const int64_t FN1 = hh_F(N - 1, NBW);
    const bool colok = col0 + lane < a.nev;
    float *const cb = a.q + (colok ? col0 + lane : 0) * a.ldq * EW;

    int64_t pk = 0, pb = bhi;                           // staging cursor: block it + NS - LAG
    auto advance = [&]() {
        if (pb > pk * C::NB8) {
            --pb;
        } else {
            ++pk;
            pb = bhi;
        }
    };
    for (int i = 0; i < NS - LAG; ++i) {
        if (member == 0 && pk < K0) f32_stage<C>(a, ring + i * C::STAGE_FLOATS, bar_full + 8 * i, pk, pb, FN1, lane);
        advance();
    }
    float xr[W], xi[CPLX ? W : 8];
    // incoming rows travel through the warp's private shared-memory ring, DQ tiles ahead of their use: no
    // register waits on a load in flight (with a register prefetch one block ahead a quarter of all samples
    // sat on the first use of the loaded rows: one block of FFMAs is about one DRAM round trip)
    float *qring = reinterpret_cast<float *>(smem + C::OFF_Q) + (size_t)member * C::NSQ * C::QTILE;
    uint32_t it = 0;
    int duty = 0;
    for (int64_t k = 0; k < K0; ++k) {
        const int64_t blo = k * C::NB8;
        int qin = 0, qout = 0;                          // ring slots of the tile fetched next / taken next
        auto fetch = [&](int64_t b) {                   // tile of block b (none below the chain: zeros)
            f32_fetch8<CPLX>(a, cb, colok && b >= blo, b << 3, qring + qin * C::QTILE, lane);
            cp_async_commit();
            qin = (qin + 1) & (C::NSQ - 1);
        };
        auto take = [&]() {                             // the oldest tile in flight into window offsets 0 .. 7
            asm volatile("cp.async.wait_group %0;" ::"n"(C::DQ - 1) : "memory");
            f32_take8<CPLX>(qring + qout * C::QTILE, lane, xr, xi);
            qout = (qout + 1) & (C::NSQ - 1);
        };
#pragma unroll
        for (int w = 0; w < W; ++w) {
            xr[w] = 0.0f;
            if (CPLX) xi[w] = 0.0f;
        }
#pragma unroll
        for (int i = 0; i < C::DQ; ++i) fetch(bhi - i);
        take();
        for (int64_t b = bhi; b >= blo; --b) {
            if (duty == member && pk < K0) {
                const uint32_t st = (it + NS - LAG) & (NS - 1);
                if (it >= (uint32_t)LAG) mbar_wait(bar_empty + 8 * st, ((it - LAG) >> C::LGNS) & 1);
                f32_stage<C>(a, ring + st * C::STAGE_FLOATS, bar_full + 8 * st, pk, pb, FN1, lane);
            }
            advance();
            duty = (duty + 1 == nmem) ? 0 : duty + 1;
            fetch(b - C::DQ);

            const uint32_t st = it & (NS - 1);
            mbar_wait(bar_full + 8 * st, (it >> C::LGNS) & 1);
            const float *V = ring + st * C::STAGE_FLOATS;
            // reflectors 0 .. 6; then the rows on top (offsets nbw .. nbw+7 = rows 8b+nbw ..) are final and
            // retire; reflector 7 writes its result 8 registers further on
            f32_block_step<C, 0, 7>(xr, xi, V, V + C::V_FLOATS);
            f32_store8<CPLX>(a, cb, colok, (b << 3) + NBW, xr + NBW, xi + (CPLX ? NBW : 0));
            f32_block_step<C, 7, 8>(xr, xi, V, V + C::V_FLOATS);
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty + 8 * st);
            take();                                     // rows of block b-1
            ++it;
        }
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        // chain end: offsets 8 .. W-1 hold rows 8 blo .. 8 blo + nbw - 1
#pragma unroll
        for (int t = 0; t < C::NB8; ++t)
            f32_store8<CPLX>(a, cb, colok, (blo << 3) + 8 * t, xr + 8 + 8 * t, xi + (CPLX ? 8 + 8 * t : 0));
    }
}

// ---- the kernel: CTA c takes strips [nstrip*c/grid, nstrip*(c+1)/grid), one per warp (at most 8) ------------
template <bool CPLX, int NBW>
__global__ void __launch_bounds__(256, 1) bt_f32_kernel(const F32Args a)
{
    using C = F32Cfg<CPLX, NBW>;
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t bar_full = smem_u32(smem + C::OFF_BAR);
    const uint32_t bar_empty = bar_full + C::NS * 8;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t nstrip = (a.nev + 31) >> 5;
    const int64_t strip0 = nstrip * blockIdx.x / gridDim.x;
    const int nmine = (int)(nstrip * (blockIdx.x + 1) / gridDim.x - strip0);
    if (threadIdx.x == 0) {
        for (int i = 0; i < C::NS; ++i) {
            mbar_init(bar_full + 8 * i, 32);           // 32 cp.async arrivals (one per lane of the staging warp)
            mbar_init(bar_empty + 8 * i, (uint32_t)nmine);
        }
        mbar_fence_init();
    }
    __syncthreads();
    if (warp >= nmine) return;
    f32_consume<C>(a, smem, lane, warp, nmine, (strip0 + warp) << 5);
}

// launch plan: a multiple of the SM count of CTAs (or one CTA per strip if there are fewer), <= 8 strips each
inline int64_t f32_grid(int64_t nev, int nsm)
{
    const int64_t nstrip = (nev + 31) >> 5;
    const int64_t waves = (nstrip + (int64_t)nsm * 8 - 1) / ((int64_t)nsm * 8);
    const int64_t grid = (int64_t)nsm * waves;
    return grid < nstrip ? grid : nstrip;
}

template <bool CPLX, int NBW>
cudaError_t launch_f32(int64_t N, int64_t nev, const float *hh_v, const float *hh_tau, float *q, int64_t ldq, int align16,
                       int nsm, cudaStream_t st)
{
    using C = F32Cfg<CPLX, NBW>;
    auto kern = bt_f32_kernel<CPLX, NBW>;
    cudaError_t e = set_max_smem((const void *)kern, C::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    F32Args a;
    a.N = N;
    a.nev = nev;
    a.ldq = ldq;
    a.hh_v = hh_v;
    a.hh_tau = hh_tau;
    a.q = q;
    a.align16 = align16;
    kern<<<(unsigned)f32_grid(nev, nsm), 256, C::SMEM_BYTES, st>>>(a);
    return cudaGetLastError();
}

}  // namespace elpa2bt
