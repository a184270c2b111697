// elpa2_bt.cu -- C-ABI entry points of include/elpa2_bt.h: argument validation, launch planning,
// host-buffer wrapper.  All arithmetic of the path is in the kernels (bt_wy.cuh / bt_wyz.cuh: the
// default, compact-WY on the FP64 tensor cores, real / complex; bt_shift.cuh: variant 2, one
// reflector at a time in a register window, DFMA; bt_simple.cuh: variant 1, plain A/B baseline).
// No torch types, no CPU fallback.
#include "../../include/elpa2_bt.h"

#include <cuda_runtime.h>

#include <atomic>
#include <cstdlib>
#include <mutex>

#include "bt_shift.cuh"
#include "bt_simple.cuh"
#include "bt_wy.cuh"
#include "bt_wyz.cuh"
#include "bc_chase.cuh"
#include "bt_b2f.cuh"
#include "bt_b2fz.cuh"
#include "bt_f32.cuh"

using namespace elpa2bt;

#ifndef ELPA2_BT_UNROLL
#define ELPA2_BT_UNROLL 2
#endif

namespace {

// library state is per calling thread (variant selector, launch counter) or per device (SM count,
// scratch pool, kernel attributes): no call changes what another thread's or another device's call does
thread_local int g_variant = 0;
thread_local int g_last_launches = 0;
thread_local int g_force_P = 0;     // testing aid (elpa2_bt_set_chain_parallel): warps per slab, 0 = planned
constexpr int MAX_DEV = 64;
std::mutex g_mu;        // host-buffer entry point (its cached device scratch)
std::mutex g_pool_mu;   // creation of the scratch pool

// Widths (R13, "multiples of 32"): the back-transformation is instantiated for every
// multiple of 32 up to 256 (real) / 160 (complex: the planar window of one slab must fit in 255
// registers); the bulge chase and variant 2 for the recommended 32, 64, 128.
bool bt_width_ok(int nbw, bool cplx) { return nbw >= 32 && (nbw & 31) == 0 && nbw <= (cplx ? 160 : 256); }
bool pow2_width_ok(int nbw) { return nbw == 32 || nbw == 64 || nbw == 128; }

// expands to `case w: stmt(w)` for the instantiated widths
#define ELPA2_REAL_WIDTHS(X) X(32) X(64) X(96) X(128) X(160) X(192) X(224) X(256)
#define ELPA2_CPLX_WIDTHS(X) X(32) X(64) X(96) X(128) X(160)
// FP32 (bt_f32.cuh): the window of one column sits in one lane's registers
bool f32_width_ok(int nbw, bool cplx) { return nbw >= 32 && (nbw & 31) == 0 && nbw <= (cplx ? 64 : 128); }

int current_device()
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEV) return 0;
    return dev;
}

int sm_count()
{
    static std::atomic<int> n[MAX_DEV];
    const int dev = current_device();
    int v = n[dev].load(std::memory_order_relaxed);
    if (v == 0) {
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) return 148;
        n[dev].store(v, std::memory_order_relaxed);
    }
    return v;
}

// the shift kernel: 7 consumer warps + 1 producer warp = 256 threads, so that each thread may use
// up to 255 registers (the window, CPL columns x RL rows per lane, takes 128 of them)
template <bool CPLX, int NBW, int CPL>
cudaError_t launch_shift(int64_t N, int64_t nev, const double *hh_v, const double *hh_tau, double *q,
                         int64_t ldq, int align16, cudaStream_t st)
{
    using C = ShiftCfg<CPLX, NBW, CPL>;
    constexpr int MAXT = 256;
    auto kern = bt_shift_kernel<CPLX, NBW, CPL, MAXT, ELPA2_BT_UNROLL>;
    constexpr int NWMAX = MAXT / 32 - 1;
    {
        cudaError_t e = set_max_smem((const void *)kern, (int)C::smem_bytes(NWMAX));
        if (e != cudaSuccess) return e;
    }
    const int64_t units = (nev + C::CW - 1) / C::CW;
    const int64_t nsm = sm_count();
    const int64_t waves = (units + nsm * NWMAX - 1) / (nsm * NWMAX);
    int64_t grid = nsm * waves;                       // a multiple of the SM count ...
    if (grid > units) grid = units;                   // ... unless there are fewer warp-units
    const int64_t nw = (units + grid - 1) / grid;     // the kernel splits the units evenly over CTAs
    WinArgs a;
    a.N = N;
    a.nev = nev;
    a.ldq = ldq;
    a.hh_v = hh_v;
    a.hh_tau = hh_tau;
    a.q = q;
    a.nw = (int)nw;
    a.align16 = align16;
    kern<<<(unsigned)grid, (unsigned)((nw + 1) * 32), C::smem_bytes((int)nw), st>>>(a);
    return cudaGetLastError();
}

// stream-ordered scratch for the -T factors of the WY kernel: a private memory pool that keeps
// what it has allocated (release threshold = max), so that in steady state a call allocates
// nothing new and never synchronises the host
cudaMemPool_t g_pool[MAX_DEV] = {};     // one per device, written under g_pool_mu

cudaMemPool_t scratch_pool(cudaError_t *err)
{
    int dev = 0;
    *err = cudaGetDevice(&dev);
    if (*err != cudaSuccess) return nullptr;
    if (dev < 0 || dev >= MAX_DEV) {
        *err = cudaErrorInvalidDevice;
        return nullptr;
    }
    std::lock_guard<std::mutex> lock(g_pool_mu);
    cudaMemPool_t &pool = g_pool[dev];
    if (pool) return pool;
    cudaMemPoolProps props = {};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    cudaMemPool_t p = nullptr;
    *err = cudaMemPoolCreate(&p, &props);
    if (*err != cudaSuccess) return nullptr;
    uint64_t keep = UINT64_MAX;
    cudaMemPoolSetAttribute(p, cudaMemPoolAttrReleaseThreshold, &keep);
    pool = p;
    return pool;
}

template <int NBW>
cudaError_t run_wy(int64_t N, int64_t nev, const double *hh_v, const double *hh_tau, double *q, int64_t ldq,
                   int align16, cudaStream_t st, int force_P = 0, const WyRange &rg = WyRange())
{
    cudaError_t e;
    cudaMemPool_t pool = scratch_pool(&e);
    if (!pool) return e;
    void *tn = nullptr;
    size_t bytes = wy_scratch_bytes<NBW>(N, nev);
    if (!rg.whole()) {
        int64_t kb, ke, bt, bb, re;
        wy_range_resolve(rg, N, NBW, kb, ke, bt, bb, re);
        if (ke <= kb) return cudaSuccess;
        bytes = wy_tn_bytes_range<NBW>(N, kb, ke) + 256;
    }
    if ((e = cudaMallocFromPoolAsync(&tn, bytes, pool, st)) != cudaSuccess) return e;
    e = launch_wy<NBW>(N, nev, hh_v, hh_tau, q, ldq, align16, sm_count(), tn, st, force_P, 0, rg);
    const cudaError_t e2 = cudaFreeAsync(tn, st);
    return e != cudaSuccess ? e : e2;
}

template <int NBW>
cudaError_t run_wyz(int64_t N, int64_t nev, const double *hh_v, const double *hh_tau, double *q, int64_t ldq,
                    cudaStream_t st, int force_P = 0, const WyRange &rg = WyRange())
{
    cudaError_t e;
    cudaMemPool_t pool = scratch_pool(&e);
    if (!pool) return e;
    void *tn = nullptr;
    size_t bytes = wyz_scratch_bytes<NBW>(N, nev);
    if (!rg.whole()) {
        int64_t kb, ke, bt, bb, re;
        wy_range_resolve(rg, N, NBW, kb, ke, bt, bb, re);
        if (ke <= kb) return cudaSuccess;
        bytes = wyz_tn_bytes_range<NBW>(N, kb, ke) + 256;
    }
    if ((e = cudaMallocFromPoolAsync(&tn, bytes, pool, st)) != cudaSuccess) return e;
    e = launch_wyz<NBW>(N, nev, hh_v, hh_tau, q, ldq, sm_count(), tn, st, force_P, rg);
    const cudaError_t e2 = cudaFreeAsync(tn, st);
    return e != cudaSuccess ? e : e2;
}

template <bool CPLX>
int run(int64_t N, int nbw, int64_t nev, const double *hh_v, const double *hh_tau, double *q, int64_t ldq,
        void *stream)
{
    constexpr int EW = CPLX ? 2 : 1;
    if (N < 0) return -1;
    if (!bt_width_ok(nbw, CPLX)) return -2;
    if (g_variant == 2 && !pow2_width_ok(nbw)) return -2;
    if (nev < 0) return -3;
    g_last_launches = 0;
    if (N <= 1 || nev == 0) return 0;
    if (!hh_v) return -4;
    if (!hh_tau) return -5;
    if (!q) return -6;
    if (ldq < N) return -7;
    if (((uintptr_t)hh_v & 15) != 0) return -4;
    if (((uintptr_t)hh_tau & (8 * EW - 1)) != 0) return -5;
    if (((uintptr_t)q & (8 * EW - 1)) != 0) return -6;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    int nlaunch = 1;
    if (g_variant == 1) {
        const unsigned grid = (unsigned)((nev + 127) / 128);
        bt_simple_kernel<CPLX><<<grid, 128, 0, st>>>(N, nbw, nev, hh_v, hh_tau, q, ldq);
        e = cudaGetLastError();
    } else if ((g_variant == 0 || g_variant == 3) && CPLX) {
        const int fp = g_force_P > 2 ? 2 : g_force_P;
        switch (nbw) {
#define X(w) case w: e = run_wyz<w>(N, nev, hh_v, hh_tau, q, ldq, st, fp); break;
            ELPA2_CPLX_WIDTHS(X)
#undef X
        default: return -2;
        }
        nlaunch = 2;
    } else if (g_variant == 0 || (g_variant == 3 && !CPLX)) {
        // variant 3: two chains per pass (pairs of warps share their slabs, hand-over through L2)
        const int align16 = (((uintptr_t)q & 15) == 0 && (ldq & 1) == 0) ? 1 : 0;
        const int fp = g_force_P ? g_force_P : (g_variant == 3 && wy_nchains(N, nbw) >= 8) ? 2 : 0;
        switch (nbw) {
#define X(w) case w: e = run_wy<w>(N, nev, hh_v, hh_tau, q, ldq, align16, st, fp); break;
            ELPA2_REAL_WIDTHS(X)
#undef X
        default: return -2;
        }
        nlaunch = 2;
    } else {
        const int align16 = CPLX ? 1 : ((((uintptr_t)q & 15) == 0 && (ldq & 1) == 0) ? 1 : 0);
        switch (nbw) {
        case 32: e = launch_shift<CPLX, 32, 2>(N, nev, hh_v, hh_tau, q, ldq, align16, st); break;
        case 64: e = launch_shift<CPLX, 64, 2>(N, nev, hh_v, hh_tau, q, ldq, align16, st); break;
        default: e = launch_shift<CPLX, 128, 2>(N, nev, hh_v, hh_tau, q, ldq, align16, st); break;
        }
    }
    if (e != cudaSuccess) return (int)e;
    g_last_launches = nlaunch;
    return 0;
}

template <bool CPLX>
int run_f32(int64_t N, int nbw, int64_t nev, const float *hh_v, const float *hh_tau, float *q, int64_t ldq, void *stream)
{
    constexpr int EW = CPLX ? 2 : 1;
    if (N < 0) return -1;
    if (!f32_width_ok(nbw, CPLX)) return -2;
    if (nev < 0) return -3;
    g_last_launches = 0;
    if (N <= 1 || nev == 0) return 0;
    if (!hh_v || ((uintptr_t)hh_v & 15) != 0) return -4;
    if (!hh_tau || ((uintptr_t)hh_tau & (4 * EW - 1)) != 0) return -5;
    if (!q || ((uintptr_t)q & (4 * EW - 1)) != 0) return -6;
    if (ldq < N) return -7;
    const int align16 = (((uintptr_t)q & 15) == 0 && ((ldq * EW) & 3) == 0) ? 1 : 0;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    switch (nbw) {
    case 32: e = launch_f32<CPLX, 32>(N, nev, hh_v, hh_tau, q, ldq, align16, sm_count(), st); break;
    case 64: e = launch_f32<CPLX, 64>(N, nev, hh_v, hh_tau, q, ldq, align16, sm_count(), st); break;
    case 96: e = launch_f32<false, 96>(N, nev, hh_v, hh_tau, q, ldq, align16, sm_count(), st); break;
    default: e = launch_f32<false, 128>(N, nev, hh_v, hh_tau, q, ldq, align16, sm_count(), st); break;
    }
    if (e != cudaSuccess) return (int)e;
    g_last_launches = 1;
    return 0;
}

// row-block form: see include/elpa2_bt.h
template <bool CPLX>
int run_rows(int64_t N, int nbw, int64_t nev, const double *hh_v, const double *hh_tau, double *q_local, int64_t ldq,
             int64_t row0, int64_t nown, int64_t nloc, int64_t kb, int64_t ke, void *stream)
{
    constexpr int EW = CPLX ? 2 : 1;
    if (N < 0) return -1;
    if (!bt_width_ok(nbw, CPLX)) return -2;
    if (nev < 0) return -3;
    g_last_launches = 0;
    if (row0 < 0 || (row0 & 7) != 0 || row0 > N) return -8;
    if (nown < 0 || row0 + nown > N || (row0 + nown < N && (nown & 7) != 0)) return -9;
    const int64_t need = (row0 + nown + nbw < N ? nown + nbw : N - row0);
    if (nloc < need || row0 + nloc > N) return -10;
    if (kb < 0 || ke < kb) return -11;
    if (N <= 1 || nev == 0 || nown == 0 || ke == kb) return 0;
    if (!hh_v || ((uintptr_t)hh_v & 15) != 0) return -4;
    if (!hh_tau || ((uintptr_t)hh_tau & (8 * EW - 1)) != 0) return -5;
    if (!q_local || ((uintptr_t)q_local & (8 * EW - 1)) != 0) return -6;
    if (ldq < nloc) return -7;
    WyRange rg;
    rg.kb = kb;
    rg.ke = ke;
    rg.row0 = row0;
    rg.nown = nown;
    rg.row_end = row0 + nloc;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    if (CPLX) {
        switch (nbw) {
#define X(w) case w: e = run_wyz<w>(N, nev, hh_v, hh_tau, q_local, ldq, st, 1, rg); break;
            ELPA2_CPLX_WIDTHS(X)
#undef X
        default: return -2;
        }
    } else {
        const int align16 = (((uintptr_t)q_local & 15) == 0 && (ldq & 1) == 0) ? 1 : 0;
        switch (nbw) {
#define X(w) case w: e = run_wy<w>(N, nev, hh_v, hh_tau, q_local, ldq, align16, st, 1, rg); break;
            ELPA2_REAL_WIDTHS(X)
#undef X
        default: return -2;
        }
    }
    if (e != cudaSuccess) return (int)e;
    g_last_launches = 2;
    return 0;
}

// grow-only device scratch for the host-buffer entry point
struct Scratch {
    void *p = nullptr;
    size_t cap = 0;
    cudaError_t reserve(size_t n)
    {
        if (n <= cap) return cudaSuccess;
        if (p) cudaFree(p);
        p = nullptr;
        cap = 0;
        cudaError_t e = cudaMalloc(&p, n);
        if (e == cudaSuccess) cap = n;
        return e;
    }
} g_sv, g_st, g_sq;

// ---- allocation-free entry point (elpa2_trans_ev_band_to_full_noalloc_d) ------------------------------------
// Its scratch -- the -T factors of the Eq. 6e blocks, 32 KB per block of 64 reflectors -- lives in this
// file-scope device array instead of the stream-ordered pool: 16 MiB, held by every GPU that loads the
// library until the process exits.  In host code the array's NAME is a host-side stand-in, not a device
// address: the address comes from cudaGetSymbolAddress, once per device with that device current.
constexpr size_t NOALLOC_SCRATCH_BYTES = (size_t)16 << 20;
static __device__ __align__(256) double g_noalloc_scratch[NOALLOC_SCRATCH_BYTES / sizeof(double)];
std::mutex g_noalloc_mu;
void *g_noalloc_ptr[MAX_DEV] = {};      // device address of g_noalloc_scratch, per device

cudaError_t noalloc_scratch_ptr(void **out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAX_DEV) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        g_noalloc_ptr[dev] = p;
    }
    *out = g_noalloc_ptr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" {

int elpa2_trans_ev_tridi_to_band_d(int64_t N, int nbw, int64_t nev, const double *hh_v, const double *hh_tau,
                                   double *q, int64_t ldq, void *stream)
{
    return run<false>(N, nbw, nev, hh_v, hh_tau, q, ldq, stream);
}

int elpa2_trans_ev_tridi_to_band_z(int64_t N, int nbw, int64_t nev, const void *hh_v, const void *hh_tau,
                                   void *q, int64_t ldq, void *stream)
{
    return run<true>(N, nbw, nev, (const double *)hh_v, (const double *)hh_tau, (double *)q, ldq, stream);
}

int elpa2_trans_ev_tridi_to_band_s(int64_t N, int nbw, int64_t nev, const float *hh_v, const float *hh_tau,
                                   float *q, int64_t ldq, void *stream)
{
    return run_f32<false>(N, nbw, nev, hh_v, hh_tau, q, ldq, stream);
}

int elpa2_trans_ev_tridi_to_band_c(int64_t N, int nbw, int64_t nev, const void *hh_v, const void *hh_tau,
                                   void *q, int64_t ldq, void *stream)
{
    return run_f32<true>(N, nbw, nev, (const float *)hh_v, (const float *)hh_tau, (float *)q, ldq, stream);
}

int elpa2_trans_ev_tridi_to_band_host32(int is_complex, int64_t N, int nbw, int64_t nev, const void *hh_v,
                                        const void *hh_tau, void *q, int64_t ldq)
{
    const size_t esz = is_complex ? 8 : 4;
    if (N < 0) return -1;
    if (!f32_width_ok(nbw, is_complex != 0)) return -2;
    if (nev < 0) return -3;
    if (N <= 1 || nev == 0) { g_last_launches = 0; return 0; }
    if (!hh_v) return -4;
    if (!hh_tau) return -5;
    if (!q) return -6;
    if (ldq < N) return -7;
    std::lock_guard<std::mutex> lock(g_mu);
    const size_t G = (size_t)elpa2_hh_count(N, nbw);
    const size_t bv = G * nbw * esz, bt = G * esz, bq = (size_t)ldq * nev * esz;
    cudaError_t e;
    if ((e = g_sv.reserve(bv)) != cudaSuccess) return (int)e;
    if ((e = g_st.reserve(bt)) != cudaSuccess) return (int)e;
    if ((e = g_sq.reserve(bq)) != cudaSuccess) return (int)e;
    if ((e = cudaMemcpyAsync(g_sv.p, hh_v, bv, cudaMemcpyHostToDevice, 0)) != cudaSuccess) return (int)e;
    if ((e = cudaMemcpyAsync(g_st.p, hh_tau, bt, cudaMemcpyHostToDevice, 0)) != cudaSuccess) return (int)e;
    if ((e = cudaMemcpyAsync(g_sq.p, q, bq, cudaMemcpyHostToDevice, 0)) != cudaSuccess) return (int)e;
    int rc = is_complex ? run_f32<true>(N, nbw, nev, (const float *)g_sv.p, (const float *)g_st.p, (float *)g_sq.p, ldq, 0)
                        : run_f32<false>(N, nbw, nev, (const float *)g_sv.p, (const float *)g_st.p, (float *)g_sq.p, ldq, 0);
    if (rc != 0) return rc;
    if ((e = cudaMemcpyAsync(q, g_sq.p, bq, cudaMemcpyDeviceToHost, 0)) != cudaSuccess) return (int)e;
    if ((e = cudaStreamSynchronize(0)) != cudaSuccess) return (int)e;
    return 0;
}

int elpa2_trans_ev_tridi_to_band_rows_d(int64_t N, int nbw, int64_t nev, const double *hh_v, const double *hh_tau,
                                        double *q_local, int64_t ldq, int64_t row0, int64_t nown, int64_t nloc,
                                        int64_t kb, int64_t ke, void *stream)
{
    return run_rows<false>(N, nbw, nev, hh_v, hh_tau, q_local, ldq, row0, nown, nloc, kb, ke, stream);
}

int elpa2_trans_ev_tridi_to_band_rows_z(int64_t N, int nbw, int64_t nev, const void *hh_v, const void *hh_tau,
                                        void *q_local, int64_t ldq, int64_t row0, int64_t nown, int64_t nloc,
                                        int64_t kb, int64_t ke, void *stream)
{
    return run_rows<true>(N, nbw, nev, (const double *)hh_v, (const double *)hh_tau, (double *)q_local, ldq, row0, nown,
                          nloc, kb, ke, stream);
}

int elpa2_trans_ev_tridi_to_band_host(int is_complex, int64_t N, int nbw, int64_t nev, const void *hh_v,
                                      const void *hh_tau, void *q, int64_t ldq)
{
    const size_t esz = is_complex ? 16 : 8;
    if (N < 0) return -1;
    if (!bt_width_ok(nbw, is_complex != 0)) return -2;
    if (nev < 0) return -3;
    if (N <= 1 || nev == 0) { g_last_launches = 0; return 0; }
    if (!hh_v) return -4;
    if (!hh_tau) return -5;
    if (!q) return -6;
    if (ldq < N) return -7;
    std::lock_guard<std::mutex> lock(g_mu);
    const size_t G = (size_t)elpa2_hh_count(N, nbw);
    const size_t bv = G * nbw * esz, bt = G * esz, bq = (size_t)ldq * nev * esz;
    cudaError_t e;
    if ((e = g_sv.reserve(bv)) != cudaSuccess) return (int)e;
    if ((e = g_st.reserve(bt)) != cudaSuccess) return (int)e;
    if ((e = g_sq.reserve(bq)) != cudaSuccess) return (int)e;
    if ((e = cudaMemcpyAsync(g_sv.p, hh_v, bv, cudaMemcpyHostToDevice, 0)) != cudaSuccess) return (int)e;
    if ((e = cudaMemcpyAsync(g_st.p, hh_tau, bt, cudaMemcpyHostToDevice, 0)) != cudaSuccess) return (int)e;
    if ((e = cudaMemcpyAsync(g_sq.p, q, bq, cudaMemcpyHostToDevice, 0)) != cudaSuccess) return (int)e;
    int rc = is_complex ? run<true>(N, nbw, nev, (const double *)g_sv.p, (const double *)g_st.p, (double *)g_sq.p, ldq, 0)
                        : run<false>(N, nbw, nev, (const double *)g_sv.p, (const double *)g_st.p, (double *)g_sq.p, ldq, 0);
    if (rc != 0) return rc;
    if ((e = cudaMemcpyAsync(q, g_sq.p, bq, cudaMemcpyDeviceToHost, 0)) != cudaSuccess) return (int)e;
    if ((e = cudaStreamSynchronize(0)) != cudaSuccess) return (int)e;
    return 0;
}

int elpa2_bulge_chase_d(int64_t N, int nbw, double *ab, double *hh_v, double *hh_tau, double *d, double *e,
                        void *stream)
{
    if (N < 0) return -1;
    if (!pow2_width_ok(nbw)) return -2;
    g_last_launches = 0;
    if (N == 0) return 0;
    if (!ab) return -3;
    if (N >= 2 && !hh_v) return -4;
    if (N >= 2 && !hh_tau) return -5;
    if (!d) return -6;
    if (N >= 2 && !e) return -7;
    if (((uintptr_t)ab & 7) != 0) return -3;
    if (((uintptr_t)hh_v & 7) != 0) return -4;
    if (((uintptr_t)hh_tau & 7) != 0) return -5;
    cudaStream_t st = (cudaStream_t)stream;
    int64_t nl = 0;
    cudaError_t err;
    // persistent kernel unless ELPA2_BC_WAVEFRONT=1 asks for one launch per wavefront; its
    // per-sweep progress counters come from the stream-ordered scratch pool
    static const bool wavefront_only = [] { const char *v = getenv("ELPA2_BC_WAVEFRONT"); return v && v[0] == '1'; }();
    uint32_t *prog = nullptr;
    if (N >= 2 && !wavefront_only) {
        cudaMemPool_t pool = scratch_pool(&err);
        if (!pool) return (int)err;
        if ((err = cudaMallocFromPoolAsync((void **)&prog, (size_t)2 * N * sizeof(uint32_t), pool, st)) != cudaSuccess) return (int)err;
        if ((err = cudaMemsetAsync(prog, 0, (size_t)2 * N * sizeof(uint32_t), st)) != cudaSuccess) {
            cudaFreeAsync(prog, st);
            return (int)err;
        }
    }
    switch (nbw) {
    case 32: err = launch_bulge_chase<32>(N, ab, hh_v, hh_tau, d, e, st, &nl, prog, sm_count()); break;
    case 64: err = launch_bulge_chase<64>(N, ab, hh_v, hh_tau, d, e, st, &nl, prog, sm_count()); break;
    default: err = launch_bulge_chase<128>(N, ab, hh_v, hh_tau, d, e, st, &nl, prog, sm_count()); break;
    }
    if (prog) {
        const cudaError_t e2 = cudaFreeAsync(prog, st);
        if (err == cudaSuccess) err = e2;
    }
    if (err != cudaSuccess) return (int)err;
    g_last_launches = (int)(nl > 0x7fffffff ? 0x7fffffff : nl);
    return 0;
}

int elpa2_bulge_chase_z(int64_t N, int nbw, void *ab, void *hh_v, void *hh_tau, double *d, double *e, void *stream)
{
    if (N < 0) return -1;
    if (!pow2_width_ok(nbw)) return -2;
    g_last_launches = 0;
    if (N == 0) return 0;
    if (!ab) return -3;
    if (N >= 2 && !hh_v) return -4;
    if (N >= 2 && !hh_tau) return -5;
    if (!d) return -6;
    if (N >= 2 && !e) return -7;
    // interleaved complex elements are moved 16 bytes at a time (cp.async 16, 128-bit loads)
    if (((uintptr_t)ab & 15) != 0) return -3;
    if (((uintptr_t)hh_v & 15) != 0) return -4;
    if (((uintptr_t)hh_tau & 15) != 0) return -5;
    cudaStream_t st = (cudaStream_t)stream;
    int64_t nl = 0;
    cudaError_t err;
    static const bool wavefront_only = [] { const char *v = getenv("ELPA2_BC_WAVEFRONT"); return v && v[0] == '1'; }();
    uint32_t *prog = nullptr;
    if (N >= 2 && !wavefront_only) {
        cudaMemPool_t pool = scratch_pool(&err);
        if (!pool) return (int)err;
        if ((err = cudaMallocFromPoolAsync((void **)&prog, (size_t)2 * N * sizeof(uint32_t), pool, st)) != cudaSuccess) return (int)err;
        if ((err = cudaMemsetAsync(prog, 0, (size_t)2 * N * sizeof(uint32_t), st)) != cudaSuccess) {
            cudaFreeAsync(prog, st);
            return (int)err;
        }
    }
    switch (nbw) {
    case 32: err = launch_bulge_chase_z<32>(N, (zc *)ab, (zc *)hh_v, (zc *)hh_tau, d, e, st, &nl, prog, sm_count()); break;
    case 64: err = launch_bulge_chase_z<64>(N, (zc *)ab, (zc *)hh_v, (zc *)hh_tau, d, e, st, &nl, prog, sm_count()); break;
    default: err = launch_bulge_chase_z<128>(N, (zc *)ab, (zc *)hh_v, (zc *)hh_tau, d, e, st, &nl, prog, sm_count()); break;
    }
    if (prog) {
        const cudaError_t e2 = cudaFreeAsync(prog, st);
        if (err == cudaSuccess) err = e2;
    }
    if (err != cudaSuccess) return (int)err;
    g_last_launches = (int)(nl > 0x7fffffff ? 0x7fffffff : nl);
    return 0;
}

int elpa2_trans_ev_band_to_full_d(int64_t N, int nbw, int64_t nev, const double *hv, int64_t ldv, const double *tau,
                                  double *q, int64_t ldq, void *stream)
{
    if (N < 0) return -1;
    if (nbw < 16 || (nbw & 15) != 0) return -2;
    if (nev < 0) return -3;
    g_last_launches = 0;
    if (N - nbw - 1 <= 0 || nev == 0) return 0;          // no reflector: P = I
    if (!hv || ((uintptr_t)hv & 15) != 0) return -4;
    if (ldv < N || (ldv & 1) != 0) return -5;
    if (!tau || ((uintptr_t)tau & 7) != 0) return -6;
    if (!q || ((uintptr_t)q & 7) != 0) return -7;
    if (ldq < N) return -8;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    cudaMemPool_t pool = scratch_pool(&e);
    if (!pool) return (int)e;
    void *scratch = nullptr;
    if ((e = cudaMallocFromPoolAsync(&scratch, b2f_scratch_bytes(N, nbw), pool, st)) != cudaSuccess) return (int)e;
    const int align16 = (((uintptr_t)q & 15) == 0 && (ldq & 1) == 0) ? 1 : 0;
    e = launch_b2f(N, nbw, nev, hv, ldv, tau, q, ldq, align16, sm_count(), scratch, st);
    const cudaError_t e2 = cudaFreeAsync(scratch, st);
    if (e != cudaSuccess) return (int)e;
    if (e2 != cudaSuccess) return (int)e2;
    g_last_launches = 2;
    return 0;
}

int elpa2_trans_ev_band_to_full_z(int64_t N, int nbw, int64_t nev, const void *hv, int64_t ldv, const void *tau,
                                  void *q, int64_t ldq, void *stream)
{
    if (N < 0) return -1;
    if (nbw < 16 || (nbw & 15) != 0) return -2;
    if (nev < 0) return -3;
    g_last_launches = 0;
    if (N - nbw - 1 <= 0 || nev == 0) return 0;          // no reflector: P = I
    if (!hv || ((uintptr_t)hv & 15) != 0) return -4;
    if (ldv < N) return -5;
    if (!tau || ((uintptr_t)tau & 15) != 0) return -6;
    if (!q || ((uintptr_t)q & 15) != 0) return -7;
    if (ldq < N) return -8;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    cudaMemPool_t pool = scratch_pool(&e);
    if (!pool) return (int)e;
    void *scratch = nullptr;
    if ((e = cudaMallocFromPoolAsync(&scratch, b2fz_scratch_bytes(N, nbw), pool, st)) != cudaSuccess) return (int)e;
    e = launch_b2fz(N, nbw, nev, (const double *)hv, ldv, (const double *)tau, (double *)q, ldq, sm_count(), scratch, st);
    const cudaError_t e2 = cudaFreeAsync(scratch, st);
    if (e != cudaSuccess) return (int)e;
    if (e2 != cudaSuccess) return (int)e2;
    g_last_launches = 2;
    return 0;
}

int64_t elpa2_noalloc_scratch_bytes(void) { return (int64_t)NOALLOC_SCRATCH_BYTES; }

int elpa2_trans_ev_band_to_full_noalloc_d(int64_t N, int nbw, int64_t nev, const double *hv, int64_t ldv,
                                          const double *tau, double *q, int64_t ldq, void *stream)
{
    if (N < 0) return -1;
    if (nbw < 16 || (nbw & 15) != 0) return -2;
    if (nev < 0) return -3;
    g_last_launches = 0;
    if (N - nbw - 1 <= 0 || nev == 0) return 0;          // no reflector: P = I
    if (b2f_scratch_bytes(N, nbw) > NOALLOC_SCRATCH_BYTES) return -20;   // more blocks than the static scratch holds
    if (!hv || ((uintptr_t)hv & 15) != 0) return -4;
    if (ldv < N || (ldv & 1) != 0) return -5;
    if (!tau || ((uintptr_t)tau & 7) != 0) return -6;
    if (!q || ((uintptr_t)q & 7) != 0) return -7;
    if (ldq < N) return -8;
    void *scratch = nullptr;
    cudaError_t e = noalloc_scratch_ptr(&scratch);
    if (e != cudaSuccess) return (int)e;
    const int align16 = (((uintptr_t)q & 15) == 0 && (ldq & 1) == 0) ? 1 : 0;
    // the prepass overwrites every entry of the -T factors this call reads: nothing has to start at zero
    e = launch_b2f(N, nbw, nev, hv, ldv, tau, q, ldq, align16, sm_count(), scratch, (cudaStream_t)stream);
    if (e != cudaSuccess) return (int)e;
    g_last_launches = 2;
    return 0;
}

int elpa2_trans_ev_band_to_full_host(int is_complex, int64_t N, int nbw, int64_t nev, const void *hv, int64_t ldv,
                                     const void *tau, void *q, int64_t ldq)
{
    const size_t esz = is_complex ? 16 : 8;
    if (N < 0) return -2;
    if (nbw < 16 || (nbw & 15) != 0) return -3;
    if (nev < 0) return -4;
    const int64_t Nv = N - nbw - 1;
    if (Nv <= 0 || nev == 0) { g_last_launches = 0; return 0; }
    if (!hv) return -5;
    if (ldv < N || (!is_complex && (ldv & 1) != 0)) return -6;
    if (!tau) return -7;
    if (!q) return -8;
    if (ldq < N) return -9;
    std::lock_guard<std::mutex> lock(g_mu);
    const size_t bv = (size_t)ldv * Nv * esz, bt = (size_t)Nv * esz, bq = (size_t)ldq * nev * esz;
    cudaError_t e;
    if ((e = g_sv.reserve(bv)) != cudaSuccess) return (int)e;
    if ((e = g_st.reserve(bt)) != cudaSuccess) return (int)e;
    if ((e = g_sq.reserve(bq)) != cudaSuccess) return (int)e;
    if ((e = cudaMemcpyAsync(g_sv.p, hv, bv, cudaMemcpyHostToDevice, 0)) != cudaSuccess) return (int)e;
    if ((e = cudaMemcpyAsync(g_st.p, tau, bt, cudaMemcpyHostToDevice, 0)) != cudaSuccess) return (int)e;
    if ((e = cudaMemcpyAsync(g_sq.p, q, bq, cudaMemcpyHostToDevice, 0)) != cudaSuccess) return (int)e;
    const int rc = is_complex ? elpa2_trans_ev_band_to_full_z(N, nbw, nev, g_sv.p, ldv, g_st.p, g_sq.p, ldq, 0)
                              : elpa2_trans_ev_band_to_full_d(N, nbw, nev, (const double *)g_sv.p, ldv,
                                                              (const double *)g_st.p, (double *)g_sq.p, ldq, 0);
    if (rc != 0) return rc < 0 ? rc - 1 : rc;            // argument positions shift by one (is_complex)
    if ((e = cudaMemcpyAsync(q, g_sq.p, bq, cudaMemcpyDeviceToHost, 0)) != cudaSuccess) return (int)e;
    if ((e = cudaStreamSynchronize(0)) != cudaSuccess) return (int)e;
    return 0;
}

int64_t elpa2_hh_count(int64_t N, int nbw)
{
    if (nbw < 1 || N < 2) return 0;
    return hh_F(N - 1, nbw);
}

int64_t elpa2_hh_offset(int64_t N, int nbw, int64_t s)
{
    if (nbw < 1 || N < 2 || s < 0 || s > N - 1) return -1;
    return hh_off(N, nbw, s);
}

int elpa2_hh_blocks(int64_t N, int nbw, int64_t s)
{
    if (nbw < 1 || N < 2 || s < 0 || s > N - 2) return 0;
    return (int)((N - 1 - s + nbw - 1) / nbw);
}

int64_t elpa2_hh_lengths(int64_t N, int nbw, int32_t *out, int64_t cap)
{
    if (nbw < 1 || N < 2) return 0;
    const int64_t G = hh_F(N - 1, nbw);
    if (!out) return G;
    int64_t g = 0;
    for (int64_t s = 0; s <= N - 2; ++s) {
        const int64_t K = (N - 1 - s + nbw - 1) / nbw;
        for (int64_t k = 0; k < K; ++k, ++g) {
            if (g >= cap) return G;
            const int64_t rest = N - 1 - s - k * nbw;      // rows r0 .. N-1
            out[g] = (int32_t)(rest < nbw ? rest : nbw);
        }
    }
    return G;
}

int elpa2_bt_plan(int is_complex, int64_t N, int nbw, int64_t nev, int n_sm, int64_t out[6])
{
    if (N < 0) return -2;
    if (!bt_width_ok(nbw, is_complex != 0)) return -3;
    if (nev < 0) return -4;
    if (n_sm < 1) return -5;
    if (!out) return -6;
    for (int i = 0; i < 6; ++i) out[i] = 0;
    if (N <= 1 || nev == 0) return 0;
    const int fp = g_force_P ? g_force_P : (g_variant == 3 && !is_complex && wy_nchains(N, nbw) >= 8) ? 2 : 0;
    const WyPlan pl = wy_plan(is_complex != 0, nbw, N, nev, n_sm, fp, is_complex ? 8 : 0);
    size_t scratch = 0;
    switch (nbw + (is_complex ? 1 : 0)) {
#define X(w) case w: scratch = wy_scratch_bytes<w>(N, nev); break;
        ELPA2_REAL_WIDTHS(X)
#undef X
#define X(w) case w + 1: scratch = wyz_scratch_bytes<w>(N, nev); break;
        ELPA2_CPLX_WIDTHS(X)
#undef X
    }
    out[0] = pl.grid;
    out[1] = pl.nwarps;
    out[2] = pl.P;
    out[3] = pl.nslab;
    out[4] = pl.per_cta;
    out[5] = (int64_t)scratch;
    return 0;
}

int elpa2_bt_release_scratch(void)
{
    cudaError_t first = cudaSuccess;
    {
        std::lock_guard<std::mutex> lock(g_mu);
        for (Scratch *s : {&g_sv, &g_st, &g_sq}) {
            if (s->p) {
                const cudaError_t e = cudaFree(s->p);
                if (first == cudaSuccess) first = e;
            }
            s->p = nullptr;
            s->cap = 0;
        }
    }
    std::lock_guard<std::mutex> lock(g_pool_mu);
    for (int dev = 0; dev < MAX_DEV; ++dev)
        if (g_pool[dev]) {
            const cudaError_t e = cudaMemPoolTrimTo(g_pool[dev], 0);
            if (first == cudaSuccess) first = e;
        }
    return (int)first;
}

int elpa2_bt_last_launch_count(void) { return g_last_launches; }

int elpa2_bt_set_variant(int variant)
{
    if (variant < 0 || variant > 3) return -1;
    const int old = g_variant;
    g_variant = variant;
    return old;
}

int elpa2_bt_set_chain_parallel(int P)
{
    if (P != 0 && P != 1 && P != 2 && P != 4) return -1;
    const int old = g_force_P;
    g_force_P = P;
    return old;
}

const char *elpa2_bt_version(void) { return "elpa2-bt-b200 0.1 (sm_100a)"; }

}  // extern "C"
