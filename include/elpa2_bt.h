/*
 * elpa2_bt.h -- C ABI of the B200-native stage-2 eigenvector back-transformation of ELPA2
 * (arxiv 2002.10991, Eq. 6d; citations are "PAPER.md:<line>" of the extracted paper text,
 * "R<n>" are the readings listed in DESIGN.md).
 *
 * The operation (Eq. 6d, Eq. 8): given the Householder
 * reflectors H(s,k) = I - tau v v^H produced by bulge-chasing a band matrix of semi-bandwidth nbw
 * to tridiagonal form, overwrite the N x nev block q of tridiagonal-basis
 * eigenvectors with
 *
 *      q  <-  H(0,0) H(0,1) ... H(0,K(0)-1) H(1,0) ... H(N-2,0) q ,
 *
 * i.e. the reflector generated LAST is applied FIRST ("the reverse of the order in which they
 * are generated").  tau is used as stored (not conjugated); the dot product
 * is v^H x (R2).  Sweep s = 0..N-2 (the paper's stage i = s+1) has K(s) = ceil((N-1-s)/nbw)
 * chase blocks k (the paper's sweep j = k+1); reflector (s,k) acts on rows
 * r0 = s+1+k*nbw .. min(s+(k+1)*nbw, N-1) (0-based) (R1, R3).
 *
 * Reflector layout (sweep-major, generation order; "stored in a separate array"):
 *   slot g(s,k) = elpa2_hh_offset(N,nbw,s) + k;   tau at hh_tau[g];   v at hh_v[g*nbw + r],
 *   r = 0..nbw-1, with hh_v[g*nbw] == 1 stored explicitly and entries r >= L equal to ZERO (R8).
 *   tau == 0 marks an identity slot.  The producer guarantees v[0] == 1 and the zero padding.
 *
 * q: column-major, element (r, j) at q[r + j*ldq], 0 <= r < N, 0 <= j < nev, updated in place.
 * Complex data is interleaved (re, im) doubles (C99 double complex / std::complex<double>).
 *
 * Ownership and execution: the caller owns every buffer.  hh_v, hh_tau and q are DEVICE pointers
 * valid on the current CUDA device; hh_* are read-only.  The call enqueues work on `stream`
 * (a cudaStream_t passed as void*; NULL = the legacy default stream), returns without
 * synchronising the host (keep data on the device, no implicit synchronisation).
 * The default variant takes its scratch (one (nbw+8) x 8 matrix per block of 8 reflectors, about
 * N^2/(16 nbw) blocks: 0.55 N^2 doubles real, 1.2 N^2 doubles complex, i.e. 4.8 GB for N = 32768
 * real) from a stream-ordered CUDA memory pool private to the library, which keeps what it has
 * allocated: in steady state a call allocates nothing new.  There is no CPU fallback: without a CUDA device every compute call
 * fails with the cudaError_t of the launch.
 *
 * Return value: 0 on success; -i if the i-th argument (1-based: N=1, nbw=2, nev=3, hh_v=4,
 * hh_tau=5, q=6, ldq=7, stream=8) is invalid; > 0 is the cudaError_t of a failed launch.
 * Invalid: N < 0; nbw not a multiple of 32 in [32, 256] (real) / [32, 160] (complex: the planar window
 * of 8 columns must fit in 255 registers) -- PAPER.md:186: "multiples of 32 ... 32, 64, and 128 being
 * the recommended choices"; variant 2 and the bulge chase take 32, 64, 128 only; nev < 0; a NULL pointer when there is work to do; ldq < max(N,1); a q or hh_v pointer
 * that is not aligned to its element size, hh_v not 16-byte aligned (bulk-copy requirement).
 * N <= 1 or nev == 0 is success with no work.  Nothing is printed, no errno, no exceptions.
 */
#ifndef ELPA2_BT_H
#define ELPA2_BT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* FP64 real.  hh_v: G*nbw doubles, hh_tau: G doubles, q: ldq*nev doubles (all device). */
int elpa2_trans_ev_tridi_to_band_d(int64_t N, int nbw, int64_t nev,
                                   const double *hh_v, const double *hh_tau,
                                   double *q, int64_t ldq, void *stream);

/* FP64 complex, interleaved (re, im).  hh_v: G*nbw complex, hh_tau: G complex, q: ldq*nev complex
 * (all device; ldq counts complex elements). */
int elpa2_trans_ev_tridi_to_band_z(int64_t N, int nbw, int64_t nev,
                                   const void *hh_v, const void *hh_tau,
                                   void *q, int64_t ldq, void *stream);

/* Same operation with HOST buffers (pageable or pinned): copies hh_v, hh_tau and q to the device,
 * runs the kernel, copies q back and synchronises (the paper's steps 1-5).
 * Device scratch is allocated on first use and cached (grow-only).  is_complex = 0 / 1.
 * Returns like the calls above (argument positions of the _d/_z signature). */
int elpa2_trans_ev_tridi_to_band_host(int is_complex, int64_t N, int nbw, int64_t nev,
                                      const void *hh_v, const void *hh_tau,
                                      void *q, int64_t ldq);

/* the row-block form of the same operation -- the building block of the row-pipelined
 * multi-GPU variant (an eigenvector's rows spread over a process column, "at most nbw"
 * rows exchanged with the neighbour per step).  The caller owns the rows
 * [row0, row0 + nown) of q (row0 a multiple of 8; nown a multiple of 8 unless the block ends at row N)
 * and passes q_local, which holds the rows [row0, row0 + nloc) of its columns, nloc >= min(nown + nbw,
 * N - row0): the owned rows followed by the <= nbw halo rows of the neighbour below (larger row
 * indices), leading dimension ldq >= nloc.  For the chains k = kb .. ke-1 in order (chain k = the
 * reflectors (s, k) of all sweeps, applied s descending: the chain-major order of R5) the call applies the
 * reflectors whose FIRST row lies in the owned rows (in units of 8-row blocks), reading and updating the halo
 * rows they reach into.  Applying, for every chain in turn, the row blocks from the bottom of the matrix
 * to the top -- each with the halo rows as its lower neighbour left them, and handing its own first nbw
 * rows on as the upper neighbour's halo -- is the whole back-transformation, bit for bit the result of
 * elpa2_trans_ev_tridi_to_band_{d,z} (the same kernels run a sub-range of their block sequence).
 * Argument positions: N=1, nbw=2, nev=3, hh_v=4, hh_tau=5, q_local=6, ldq=7, row0=8, nown=9, nloc=10,
 * kb/ke=11; > 0 = cudaError_t.  Asynchronous on `stream`; scratch for the chains [kb, ke) only. */
int elpa2_trans_ev_tridi_to_band_rows_d(int64_t N, int nbw, int64_t nev, const double *hh_v, const double *hh_tau,
                                        double *q_local, int64_t ldq, int64_t row0, int64_t nown, int64_t nloc,
                                        int64_t kb, int64_t ke, void *stream);
int elpa2_trans_ev_tridi_to_band_rows_z(int64_t N, int nbw, int64_t nev, const void *hh_v, const void *hh_tau,
                                        void *q_local, int64_t ldq, int64_t row0, int64_t nown, int64_t nloc,
                                        int64_t kb, int64_t ke, void *stream);

/* the same operation in FP32 (R16: Eq. 8 with every product and sum in
 * float; the paper itself runs double precision only).  _s: real float; _c: complex, interleaved (re, im)
 * floats.  Same layout, same argument positions and error codes as the FP64 calls.  nbw: a multiple of
 * 32 up to 128 (real) / 64 (complex) -- the window of one column (nbw + 8 rows) sits in the registers of
 * ONE lane, applied one reflector at a time on the FP32 FMA pipe (there is no FP32 tensor-core type).
 * hh_v 16-byte aligned; q and hh_tau aligned to their element size (16-byte aligned q with ldq * element
 * size a multiple of 16 takes the vector path).  One launch, no scratch.  _host32: HOST buffers,
 * synchronous (is_complex selects _s / _c), as elpa2_trans_ev_tridi_to_band_host. */
int elpa2_trans_ev_tridi_to_band_s(int64_t N, int nbw, int64_t nev,
                                   const float *hh_v, const float *hh_tau, float *q, int64_t ldq, void *stream);
int elpa2_trans_ev_tridi_to_band_c(int64_t N, int nbw, int64_t nev,
                                   const void *hh_v, const void *hh_tau, void *q, int64_t ldq, void *stream);
int elpa2_trans_ev_tridi_to_band_host32(int is_complex, int64_t N, int nbw, int64_t nev,
                                        const void *hh_v, const void *hh_tau, void *q, int64_t ldq);

/* SURVEY.md 8(f) NEXT-1, first version: bulge chasing of a symmetric / Hermitian band matrix to
 * tridiagonal form on the device (Eq. 6b; the step is SURVEY.md 8(c) O3 / DESIGN.md
 * R3, R4, R7), emitting the reflectors in the layout the calls above consume.
 *   ab:  DEVICE, (2*nbw+1) x N doubles, column j at ab + j*(2*nbw+1), ab[(i-j) + j*(2*nbw+1)] = B[i][j]
 *        for 0 <= i-j <= nbw (lower band; rows nbw+1 .. 2*nbw of every column are room for the
 *        fill and must be zero on entry).  Overwritten with the tridiagonal matrix T.
 *   hh_v (G*nbw), hh_tau (G): DEVICE outputs, every slot written (identity slots: v = e1, tau = 0).
 *   d (N), e (N-1): DEVICE outputs, diagonal and sub-diagonal of T = Q2^T B Q2.
 * Asynchronous on `stream`, no host synchronisation.  Default schedule: ONE persistent kernel, launched
 * cooperatively (every CTA of the grid -- one per SM -- must be resident at once, because sweeps hand
 * over through per-sweep progress flags in global memory; the launch fails with a cudaError_t rather
 * than deadlock if the device cannot hold the grid), plus one small kernel that extracts d and e.  Its
 * 2N 32-bit progress counters come from the library's stream-ordered scratch pool (allocated, zeroed
 * and freed in stream order; nothing new is allocated in steady state).  With ELPA2_BC_WAVEFRONT=1 in
 * the environment (read once per process) the fallback schedule runs instead: one launch per wavefront
 * t = 3s + k of independent chase steps, about 3N launches, stream order as the only dependency, no
 * scratch.  Both schedules produce the same bits.
 * Returns 0; -i for a bad i-th argument (N=1, nbw=2, ab=3, hh_v=4, hh_tau=5, d=6, e=7; a pointer that
 * is NULL with work to do or not aligned to its element size -- 16 bytes for the complex call);
 * > 0 = cudaError_t.  N = 0: no work.  The zero fill of rows nbw+1 .. 2*nbw of `ab` is the caller's
 * duty and is not checked. */
int elpa2_bulge_chase_d(int64_t N, int nbw, double *ab, double *hh_v, double *hh_tau,
                        double *d, double *e, void *stream);
/* Complex Hermitian (interleaved (re, im); the diagonal of B real): B <- H^H B H with the complex tau
 * of R2; slot (N-2, 0) is the length-1 phase rotation of R4 that makes T real.  d, e are real. */
int elpa2_bulge_chase_z(int64_t N, int nbw, void *ab, void *hh_v, void *hh_tau,
                        double *d, double *e, void *stream);

/* the band -> full back-transformation of the eigenvectors, Eq. 6e (PAPER.md:93,
 * C = P* Y; PAPER.md:232, :302 name it a target for further optimisation).  The paper states the
 * equation only; R15 is the reading: P* = H_0 H_1 ... H_{Nv-1}, Nv = max(N - nbw - 1, 0), where
 * H_j = I - tau_j v_j v_j^H is the reflector that cleared column j below the band in the full -> band
 * reduction (Eq. 6a) and acts on rows j+nbw .. N-1.  The call overwrites
 *
 *      q  <-  H_0 ( H_1 ( ... ( H_{Nv-1} q ) ) )        (the reflector generated last is applied first)
 *
 * tau as stored (R2).  Layout: hv is column-major N x Nv with leading dimension ldv (ldv >= N, ldv even,
 * hv 16-byte aligned): column j holds v_j at rows j+nbw .. N-1, the unit head hv[j+nbw + j*ldv] == 1
 * stored explicitly, rows < j+nbw ZERO (the kernel multiplies whole tiles); tau[j], j < Nv.
 * q as above (N x nev, column-major, ldq).  All DEVICE pointers; asynchronous on `stream`; the -T factors
 * of the blocks of 64 reflectors (32 KB each) come from the library's stream-ordered scratch pool.
 * nbw: any positive multiple of 16.  Two launches (T-factor prepass + the fused DMMA kernel).
 * Returns 0; -i for a bad i-th argument (N=1, nbw=2, nev=3, hv=4, ldv=5, tau=6, q=7, ldq=8); > 0 = cudaError_t.
 * Nv == 0 or nev == 0: success, no work. */
int elpa2_trans_ev_band_to_full_d(int64_t N, int nbw, int64_t nev, const double *hv, int64_t ldv,
                                  const double *tau, double *q, int64_t ldq, void *stream);

/* Complex FP64 (interleaved (re, im) doubles; ldv, ldq count complex elements): H_j = I - tau_j v_j v_j^H
 * with tau as stored and v^H conjugated in the dot product (R2).  Same layout, same argument positions
 * and error codes; hv, tau and q must be 16-byte aligned, ldv >= N (no parity requirement).  The -T
 * factors take 64 KB per block of 64 reflectors from the scratch pool. */
int elpa2_trans_ev_band_to_full_z(int64_t N, int nbw, int64_t nev, const void *hv, int64_t ldv,
                                  const void *tau, void *q, int64_t ldq, void *stream);

/* Allocation-free variant of elpa2_trans_ev_band_to_full_d for callers that cannot allocate (CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): same operation, same arguments, same
 * kernels and results, but the -T factors go into a static 16 MiB device array inside the library
 * (elpa2_noalloc_scratch_bytes(); every GPU that loads the library holds it until the process exits)
 * instead of the stream-ordered pool.  The call issues no cudaMalloc / cudaFree / cudaMallocAsync and no
 * allocating library routine.  Limit: 32 KB per block of 64 reflectors, i.e. N - nbw - 1 <= 32768; a larger
 * problem returns -20 and launches nothing.  ALL calls share the one array (per device): calls that overlap
 * on the GPU -- two streams, or two threads -- race on it; issue them on one stream or synchronise between
 * them.  The array keeps the last call's contents; each call's prepass overwrites every entry it reads,
 * so nothing has to be cleared.  Other return codes as elpa2_trans_ev_band_to_full_d. */
int elpa2_trans_ev_band_to_full_noalloc_d(int64_t N, int nbw, int64_t nev, const double *hv, int64_t ldv,
                                          const double *tau, double *q, int64_t ldq, void *stream);
int64_t elpa2_noalloc_scratch_bytes(void);

/* Same operation with HOST buffers (pageable or pinned), synchronous: H2D of hv, tau and q, the two
 * kernels, D2H of q (what bench.py --step 6e reports as e2e).  Device scratch cached as for
 * elpa2_trans_ev_tridi_to_band_host.  Argument positions: is_complex=1, N=2, nbw=3, nev=4, hv=5, ldv=6,
 * tau=7, q=8, ldq=9. */
int elpa2_trans_ev_band_to_full_host(int is_complex, int64_t N, int nbw, int64_t nev, const void *hv,
                                     int64_t ldv, const void *tau, void *q, int64_t ldq);

/* Layout helpers (host, pure integer arithmetic; R3).  G = number of reflector slots. */
/* Length L = min(nbw, N-1-s-k*nbw) of every slot in slot order (all but the last
 * reflector of a sweep have length nbw): writes min(G, cap) entries to `out` (HOST, may be NULL to
 * query) and returns G. */
int64_t elpa2_hh_lengths(int64_t N, int nbw, int32_t *out, int64_t cap);
int64_t elpa2_hh_count(int64_t N, int nbw);
/* first slot of sweep s (s in [0, N-1]; s = N-1 gives G); -1 if out of range */
int64_t elpa2_hh_offset(int64_t N, int nbw, int64_t s);
/* K(s), 0 if s is out of range */
int elpa2_hh_blocks(int64_t N, int nbw, int64_t s);

/* Kernels launched by the last successful compute call of the calling thread (for bench.py's
 * "gpu_launches"), and a selector for A/B runs.  Both are per thread: elpa2_bt_set_variant changes what
 * later calls (and elpa2_bt_plan) of the SAME thread do and nothing else.  Variants: variant 0 = default (compact-WY
 * aggregation of 8 reflectors on the FP64 tensor cores, R6: a T-factor prepass kernel + the main
 * kernel = 2 launches; its scratch comes from a stream-ordered pool that keeps its memory),
 * 1 = plain kernel (one thread per column, literal reverse generation order), 2 = one reflector at
 * a time in a register-resident window (DFMA, 1 launch), 3 = the default path with two chains per
 * pass (real only: pairs of warps share their columns and walk alternate chains, handing rows over
 * through L2 -- half the DRAM traffic, about 8 % slower; complex runs variant 0).  Returns the
 * previous variant or -1 if `variant` is unknown. */
int elpa2_bt_last_launch_count(void);
int elpa2_bt_set_variant(int variant);
/* Testing aid (per thread): force the number P of warps that share a slab of 8 columns on interleaved
 * chains in the default variant (DESIGN.md 5.1 "chain-parallel mode"; R5 makes every P give the same
 * result): 0 = as planned, 1, 2 or 4 (complex: 4 runs as 2).  tests/test_gpu_ordering.py compares the
 * results bit for bit across P.  Returns the previous value or -1. */
int elpa2_bt_set_chain_parallel(int P);

/* Launch plan of the default variant's main kernel for a problem on a device with n_sm SMs (host, pure
 * integer arithmetic, no device needed; DESIGN.md 5.1 "Decomposition"): out = { CTAs, warps per CTA,
 * warps per slab group P (= chains walked per pass), slabs of 8 columns, most slabs per CTA, bytes
 * of scratch }.  All zero when there is no work.  Returns 0 or -i for a bad i-th argument. */
int elpa2_bt_plan(int is_complex, int64_t N, int nbw, int64_t nev, int n_sm, int64_t out[6]);

/* Gives back what the library caches: the device buffers of the host-buffer entry point and the unused
 * memory of the scratch pool (blocks still in use by enqueued calls stay).  Synchronises the device
 * (cudaFree).  Returns 0 or a cudaError_t.  Without a device and with nothing cached: 0. */
int elpa2_bt_release_scratch(void);

const char *elpa2_bt_version(void);

/* Measurement aid (synchronous; allocates and frees a small device buffer): sustained FP64 ALU
 * throughput of the current device in TFLOP/s, the denominator of the "alu" roofline.
 * kind 0 = DFMA, 1 = DMMA (mma.sync m8n8k4 f64), 2 = DMMA on even warps + DFMA on odd warps.
 * Each launch runs `iters` x 64 FMA per thread on 4 x 512 threads per SM; `reps` launches are
 * timed with CUDA events.  Returns 0, -1 on a bad argument, or a cudaError_t. */
int elpa2_bt_probe_fp64(int kind, int iters, int reps, double *tflops);

#ifdef __cplusplus
}
#endif
#endif /* ELPA2_BT_H */
