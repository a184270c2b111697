// bt_simple.cuh -- variant 1: the plain kernel.  One thread per column, reflectors applied in
// literal reverse generation order (s descending, k ascending), v staged in
// shared memory per reflector, x read and written in global memory.  Slow by construction; kept
// as the in-library A/B baseline for the register-window kernel (it reaches the result by a
// different order AND a different summation tree).
#pragma once
#include "bt_common.cuh"

namespace elpa2bt {

template <bool CPLX>
__global__ void __launch_bounds__(128) bt_simple_kernel(int64_t N, int nbw, int64_t nev, const double *hh_v,
                                                         const double *hh_tau, double *q, int64_t ldq)
{
    constexpr int EW = CPLX ? 2 : 1;
    __shared__ double vs[256 * EW];                  // nbw <= 256
    __shared__ double taus[2];
    const int64_t col = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double *x = q + (col < nev ? col : 0) * ldq * EW;
    const int64_t FN1 = hh_F(N - 1, nbw);
    for (int64_t s = N - 2; s >= 0; --s) {
        const int64_t off = FN1 - hh_F(N - 1 - s, nbw);
        const int64_t K = (N - 1 - s + nbw - 1) / nbw;
        for (int64_t k = 0; k < K; ++k) {
            const int64_t g = off + k;
            const int64_t r0 = s + 1 + k * nbw;
            int64_t L = N - r0;
            L = L > nbw ? nbw : L;
            __syncthreads();
            for (int i = threadIdx.x; i < nbw * EW; i += blockDim.x) vs[i] = hh_v[g * nbw * EW + i];
            if (threadIdx.x < EW) taus[threadIdx.x] = hh_tau[g * EW + threadIdx.x];
            __syncthreads();
            const double tr = taus[0], ti = CPLX ? taus[1] : 0.0;
            if ((tr == 0.0 && ti == 0.0) || col >= nev) continue;
            double *xr = x + r0 * EW;
            if (CPLX) {
                double dr = 0.0, di = 0.0;
                for (int r = 0; r < L; ++r) {
                    const double vr = vs[2 * r], vi = vs[2 * r + 1], ar = xr[2 * r], ai = xr[2 * r + 1];
                    dr += vr * ar + vi * ai;       // conj(v) * x
                    di += vr * ai - vi * ar;
                }
                const double hr = tr * dr - ti * di, hi = tr * di + ti * dr;
                for (int r = 0; r < L; ++r) {
                    const double vr = vs[2 * r], vi = vs[2 * r + 1];
                    xr[2 * r] -= hr * vr - hi * vi;
                    xr[2 * r + 1] -= hr * vi + hi * vr;
                }
            } else {
                double d = 0.0;
                for (int r = 0; r < L; ++r) d += vs[r] * xr[r];
                const double h = tr * d;
                for (int r = 0; r < L; ++r) xr[r] -= h * vs[r];
            }
        }
    }
}

}  // namespace elpa2bt
