/*
 * fourphonon.h -- C ABI of the B200-native FourPhonon scattering-rate library (libfourphonon_b200.so).
 *
 * The library evaluates the hot path of FourPhonon_GPU (arXiv 2510.00518): three-phonon (+,-) and four-phonon
 * (++,+-,--) scattering rates of target modes lambda=(q,j) on a uniform Gamma-centred q-mesh under the RTA, plus
 * the RTA thermal conductivity.  Every step runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.
 * Operation definitions: PAPER.md (Algorithm 1; Algorithms 3-5) with the
 * formulas the paper defers to its references taken from SURVEY.md §8(c) steps 1-8 (readings in DESIGN.md §3).
 *
 * Conventions
 *   mesh N1 x N2 x N3, N = N1*N2*N3 q-points, iq = i1 + N1*(i2 + N2*i3), q = sum_mu (i_mu/N_mu) b_mu
 *   nb = 3*natoms branches, mode index lambda = iq*nb + j
 *   units: omega rad/ps, v_g Angstrom/ps, lengths Angstrom, masses u, Phi3 eV/A^3, Phi4 eV/A^4, T K,
 *          rates 1/ps, kappa W/(m K)
 *   channels: 3ph index 0 = "+" (q'' = q + q'), 1 = "-" (q'' = q - q');
 *             4ph index 0 = "++" (q''' = q + q' + q''), 1 = "+-" (q + q' - q''), 2 = "--" (q - q' - q'')
 *
 * Memory
 *   Every array argument is documented HOST or DEVICE.  Arguments marked "loc" are host or device pointers as stated
 *   by the accompanying fp_memloc value; with FP_MEM_HOST the library performs the copies itself on `stream` (these
 *   are the end-to-end entry points: host<->device traffic happens inside the call).
 *   The library never calls cudaMalloc for data: all device storage is carved out of the caller-provided `workspace`
 *   (a DEVICE allocation, 256-byte aligned, owned by the caller, which must outlive the context).  Inputs of
 *   fp_setup are copied/derived into the workspace; they are NOT borrowed and may be freed after fp_setup returns.
 *
 * Execution
 *   All kernels and copies are issued on `stream` (a cudaStream_t passed as void*, NULL = default stream).
 *   fp_setup, fp_rates3 and fp_rates4 synchronise the stream before returning (the scratch region is reused by the
 *   next super-chunk of targets, the bounded-memory loop of Algorithm 5), so on return the outputs
 *   are complete.  fp_kappa_rta with FP_MEM_DEVICE outputs is asynchronous.
 *
 * Limits
 *   natoms <= 21 (64-bit branch masks), N_mu <= 1024, N <= 2^20 q-points, lcm(N1,N2,N3) <= 4096 (phase table in shared
 *   memory).  The clusters of an IFC list are regrouped into contraction blocks (atomA, atomB, R_A - R_B mod mesh) of
 *   its last two legs; the per-row table of a list (144 bytes per block) normally lives in the shared memory of one SM,
 *   which holds about 1,400 blocks (the synthetic configs have 10-152).  An IFC3 list beyond that is still served: its
 *   table is per target, not per row, and the 3ph kernels then read it from global memory (slower per block; the
 *   remaining cap, 16 bytes of block metadata per block in shared memory, is about 12,000 blocks).  An IFC4 list beyond
 *   about 1,400 blocks is refused: fp_rates4 returns FP_ENOMEM and fp_last_error names the block count.
 *
 * Errors
 *   Every call returns FP_OK (0) or a negative code; nothing throws or aborts.  fp_last_error(ctx) (ctx may be NULL
 *   for setup failures) returns a static/ctx-owned message.
 */
#ifndef FOURPHONON_H
#define FOURPHONON_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FP_OK       0
#define FP_EINVAL  (-1)   /* bad argument / shape / value                         */
#define FP_ENOMEM  (-2)   /* workspace too small, or an IFC list with too many contraction blocks (see Limits) */
#define FP_ECUDA   (-3)   /* a CUDA runtime call or kernel failed                 */
#define FP_ESTATE  (-4)   /* call order (e.g. fp_rates4 without IFC4 at setup)    */

typedef struct fp_ctx fp_ctx;                       /* opaque, host-side handle */

typedef enum { FP_MEM_HOST = 0, FP_MEM_DEVICE = 1 } fp_memloc;

typedef struct {
    double  lattvec[9];     /* rows a1,a2,a3, Cartesian, Angstrom                                                  */
    int32_t natoms;         /* atoms per cell (positions are not needed by the rate path)                          */
} fp_crystal;

/* Anharmonic force-constant list (HOST pointers; analysed on the host at setup).
 * Cluster t is anchored at basis atom atoms[t*ord+0] in cell 0; the other ord-1 atoms sit in cells cells[t][m][0..2]. */
typedef struct {
    int64_t        n;       /* number of clusters (triplets for ord=3, quartets for ord=4)                         */
    const int32_t *atoms;   /* n*ord   basis indices (i,j,k[,l]), 0-based                                          */
    const int32_t *cells;   /* n*(ord-1)*3 integer cell offsets of j,k[,l]                                         */
    const double  *phi;     /* n*3^ord, index order alpha slowest ... last Cartesian index fastest                 */
} fp_ifc;

/* Adaptive Gaussian broadening (compute_sigma).                              */
typedef struct {
    double scale;           /* "scalebroad"; BASELINE configs use 1.0; must be > 0                                 */
    double ncut;            /* window half-width in sigma: 2.0 = PAPER.md:163; INFINITY disables the filter        */
    double sigma_const;     /* 0 -> adaptive sigma; > 0 -> this sigma (rad/ps) for every process (test mode,       */
                            /* adaptive sigma is identically 0 on 2x2x2 meshes)           */
} fp_broadening;

/* Device-time profile of the kernels launched since the last fp_profile_reset (CUDA events on the launch stream).   */
typedef struct {
    double  ms_precontract, ms_rates, ms_reduce;      /* summed launch durations, ms: per-target pre-contraction, the  */
    int64_t n_precontract, n_rates, n_reduce;         /* evaluator (k_eval_g; fused: k_rates), per-mode reduction; launches */
    int64_t rows;           /* rows ((target, channel[, lambda']) units of work: one process list and one partial sum each)  */
    int64_t candidates;     /* momentum-conserving candidates examined by the enumerator                            */
    int64_t prefiltered;    /* candidates admitted by the FP32 pre-filter (superset of the allowed ones)            */
    int64_t processes;      /* allowed processes (pinned FP64 decision) evaluated                                   */
    double  rates_flops;    /* FP64 flops of the per-process contraction (analytic model)             */
    double  ms_enum;        /* split path: summed durations of the enumerator kernel (ms_rates is then the evaluator) */
    int64_t n_enum;
    int64_t evaluated;      /* matrix elements evaluated (= processes unless the pair symmetry is in effect)          */
    int64_t list_overflows; /* split path: (row, warp) list slots that filled up (their rows were redone fused)      */
} fp_profile;

/* Bytes of workspace fp_setup needs for its resident tables plus `scratch_bytes` of per-call scratch: per-target
 * pre-contracted tables, 20 bytes per row of partial sums and -- in half of it -- the process lists of the split path
 * (4 x N x nb^2 bytes per row; a larger scratch means more rows per launch: 48 GB gives 43,668 rows at 16x16x16, nb = 6;
 * below 256 rows of lists the fused path runs instead, see fp_set_path).  ifc3/ifc4 may be NULL.  Returns 0 on invalid
 * arguments.                                                                                                          */
size_t fp_workspace_bytes(const fp_crystal *crystal, const int32_t mesh[3], const fp_ifc *ifc3, const fp_ifc *ifc4,
                          size_t scratch_bytes);

/* a1 of SURVEY.md §8(a): build the resident tables (B_mu = b_mu/N_mu, BE occupations f_lambda, mass-
 * scaled eigenvectors, mode records, Bloch phase table (a4), IFC block structure).
 *   masses   HOST natoms (u)
 *   omega    loc  N*nb            (rad/ps; the three Gamma acoustic modes must be exactly 0.0, item 8)
 *   eig      loc  N*nb*nb*2       [iq][j][3*atom+alpha][re,im]
 *   vg       loc  N*nb*3          (Angstrom/ps)
 *   ifc3, ifc4 may be NULL (then fp_rates3 / fp_rates4 return FP_ESTATE)
 * Errors: FP_EINVAL for mesh <= 0, natoms <= 0 or > 21, NaN/negative omega, 0 < omega < 1e-6*omega_max, T <= 0,
 * scale <= 0, ncut < 0, atom index out of range, lcm(N1,N2,N3) > 4096, more than 2^20 q-points; FP_ENOMEM if
 * workspace_bytes is too small.                                                                                    */
int fp_setup(const fp_crystal *crystal, const double *masses, const double *omega, const double *eig, const double *vg,
             fp_memloc mode_arrays_loc, const fp_ifc *ifc3, const fp_ifc *ifc4, const int32_t mesh[3], double T,
             const fp_broadening *broadening, void *workspace, size_t workspace_bytes, void *stream, fp_ctx **out);

/* a2+a5+a7+a8: three-phonon rates of `ntargets` target modes (Algorithms 1/3/4).
 *   targets  loc  ntargets mode indices lambda
 *   gamma    loc  ntargets*2  (+,-)  1/ps:  Gamma+ = (C3/N) sum WP+ |V+|^2,  Gamma- = (C3/N)(1/2) sum WP- |V-|^2
 *   wp       loc  ntargets*2  weighted phase space (same sums without |V|^2 and C3), nullable
 *   counts   loc  ntargets*2  number of allowed processes in the full rectangular domain (int64), nullable
 * Zero-frequency targets get 0 everywhere.  FP_EINVAL for a target index out of range.                              */
int fp_rates3(fp_ctx *ctx, const int32_t *targets, int64_t ntargets, double *gamma, double *wp, int64_t *counts,
              fp_memloc loc, void *stream);

/* a3+a6+a7+a8: four-phonon rates, channels (++,+-,--), summing only q' in [qp_begin, qp_end) (0, N = the full
 * definition).  The prefactor is always C4/N^2 so disjoint q' ranges add up to the full rate.
 *   gamma, wp: ntargets*3;  counts: ntargets*3 int64.                                                               */
int fp_rates4(fp_ctx *ctx, const int32_t *targets, int64_t ntargets, int32_t qp_begin, int32_t qp_end, double *gamma,
              double *wp, int64_t *counts, fp_memloc loc, void *stream);

/* a9: kappa^{ab} = C_kappa/(T^2 Omega N) sum_lambda f(f+1) omega^2 v^a v^b / Gamma_lambda, skipping zero modes and
 * modes with Gamma <= 0.   gamma_total loc N*nb (1/ps);  kappa loc 9 (row-major 3x3, W/(m K)).                      */
int fp_kappa_rta(fp_ctx *ctx, const double *gamma_total, double *kappa, fp_memloc loc, void *stream);

/* The same kappa for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc).  fp_kappa_rta_static calls no cudaMalloc / cudaFree and touches none of the context's workspace
 * scratch: a multi-CTA reduction (fixed summation order, so it equals fp_kappa_rta to rounding order, not bit for bit)
 * whose scratch -- the staged rates for FP_MEM_HOST, per-CTA partial sums, a ticket counter -- is ONE static device
 * array of FP_NOALLOC_MAX_MODES doubles + 5 KB (529,040 bytes), held by every GPU that loads the library until the
 * process exits.  Limit: N*nb <= FP_NOALLOC_MAX_MODES, else FP_EINVAL (fp_last_error names both numbers).  The device
 * of fp_setup must be current (FP_ESTATE otherwise).  All calls share the array: calls that overlap on the GPU (two
 * streams, two host threads, two contexts on one device) race on it; calls ordered on one stream do not.
 * FP_MEM_HOST synchronises the stream before returning; FP_MEM_DEVICE is asynchronous.                                */
#define FP_NOALLOC_MAX_MODES 65536
int fp_kappa_rta_static(fp_ctx *ctx, const double *gamma_total, double *kappa, fp_memloc loc, void *stream);

/* Debug export (not timed): the allowed-process list of one target and 3ph channel as (lambda', lambda'') pairs.
 *   pairs HOST cap*2 int32; *n receives the number of allowed processes (may exceed cap; only cap are written).
 * Order is the enumerator's (ascending q', j', j''); compare as sets.                                               */
int fp_list3(fp_ctx *ctx, int32_t target, int32_t channel, int32_t *pairs, int64_t cap, int64_t *n, void *stream);

/* Debug export: the 4ph allowed-process list of one target, channel and q' as (lambda', lambda'', lambda''') triples.
 *   triples HOST cap*3 int32.                                                                                        */
int fp_list4(fp_ctx *ctx, int32_t target, int32_t channel, int32_t qp, int32_t *triples, int64_t cap, int64_t *n,
             void *stream);

/* Per-process terms (an iterative BTE solver needs the rate of every process,
 * not only the per-mode sums).  The same lists as fp_list3 / fp_list4 -- full rectangular domain, no symmetry reuse --
 * with, for every process p, its contribution to the rate of the target in that channel:
 *   gamma_p = (C3/N) s_ch WP_p |V3_p|^2   resp.   (C4/N^2) s_ch WP_p |V4_p|^2      (1/ps; s_ch = 1, 1/2 | 1/2, 1/2, 1/6)
 * from the same pinned window decision, weights and level-2 contraction as fp_rates3 / fp_rates4, so that
 * sum_p gamma_p = Gamma^{ch}(target) (over q' = qp for fp_terms4) up to summation order.
 *   pairs / triples  HOST cap*2 / cap*3 int32 (nullable if cap == 0);  gamma_p  HOST cap doubles
 *   *n receives the number of allowed processes (may exceed cap; only cap entries are written).                       */
int fp_terms3(fp_ctx *ctx, int32_t target, int32_t channel, int32_t *pairs, double *gamma_p, int64_t cap, int64_t *n, void *stream);
int fp_terms4(fp_ctx *ctx, int32_t target, int32_t channel, int32_t qp, int32_t *triples, double *gamma_p, int64_t cap, int64_t *n,
              void *stream);

/* Execution path of fp_rates3 / fp_rates4 (same results bit for bit in counts, within rounding order in rates):
 *   FP_PATH_SPLIT_SERIAL  enumerator kernel (pre-filter, pinned FP64 decision, weights) -> process lists in half of the
 *                  scratch region -> evaluator kernel (|V|^2, row sums): Algorithms 3 and 4, both on
 *                  the device, over chunks of rows sized to the scratch, back to back on the caller's stream;
 *   FP_PATH_SPLIT  the same with two list buffers and a second (library-owned, high-priority) stream: the enumerator of
 *                  chunk k+1 runs beside the evaluator of chunk k;
 *   FP_PATH_FUSED  one kernel per chunk of targets, lists in shared memory only (needs 20 bytes of scratch per row);
 *   FP_PATH_AUTO   (default) SPLIT_SERIAL when half of the scratch holds the lists of at least 256 rows (16 bytes x
 *                  every candidate of a row), else FUSED.                                                            */
#define FP_PATH_AUTO  0
#define FP_PATH_FUSED 1
#define FP_PATH_SPLIT 2
#define FP_PATH_SPLIT_SERIAL 3
int fp_set_path(fp_ctx *ctx, int path);

/* Pair symmetry of the channels whose two free legs are both conjugated: 3ph -, 4ph +- and --.  fp_setup checks whether
 * each IFC list is invariant under the exchange of its last two legs (Phi^{abgt}(i,j,k Rk,l Rl) = Phi^{abtg}(i,j,l Rl,k Rk),
 * resp. Phi^{abg}(i,j Rj,k Rk) = Phi^{agb}(i,k Rk,j Rj), to 1e-13 of the largest entry: a derivative symmetry of every
 * physical force-constant set).  If it is, |V| and the occupation factors of those channels are symmetric under the
 * exchange of the two free legs, and the split path evaluates the matrix element of each unordered
 * pair once, taking the window decision (pinned arithmetic) and the Gaussian weight of both orderings separately: counts
 * stay bit-exact, rates change by summation order only.  fp_set_symmetry(ctx, 0) turns the reuse off; fp_get_symmetry
 * returns a bit mask of what is in effect: 1 = 3ph, 2 = 4ph.                                                         */
int fp_set_symmetry(fp_ctx *ctx, int on);
int fp_get_symmetry(const fp_ctx *ctx);

/* Time-reversal reuse over targets (PAPER.md:135-136 evaluates targets of the irreducible part
 * only).  fp_setup checks, bit for bit, that the mode arrays satisfy omega(-q,j) = omega(q,j), v(-q,j) = -v(q,j) and
 * e(-q,j) = conj(e(q,j)).  If they do, the targets (q,j) and (-q,j) of one fp_rates3 call -- or of one fp_rates4 call over
 * the whole q' range -- share their result: the library evaluates one of each pair present in `targets` and copies
 * Gamma, WP and the counts to the other (the two sums run over mirrored sets of processes with bitwise equal window
 * decisions and weights and complex-conjugate matrix elements: counts identical, rates equal to rounding order).
 * fp_set_target_symmetry(ctx, 0) turns it off; fp_get_target_symmetry returns 1 if it is in effect.                    */
int fp_set_target_symmetry(fp_ctx *ctx, int on);
int fp_get_target_symmetry(const fp_ctx *ctx);

/* Mixed precision ("FP32 where accuracy allows").  FP_PREC_MIXED evaluates the
 * per-process matrix element -- the level-2 contraction of the group path's evaluator, > 95 % of the FP64 work -- in FP32
 * (eigenvectors, the per-row table Mhat and the phases rounded to FP32, FP32 FMAs); the window decision, hence the counts,
 * the weights WP, levels 0 and 1 of the contraction and all sums stay FP64.  Gamma then carries the FP32 rounding of
 * |V|^2 (relative error ~1e-6 per process, less in the sums): it does NOT meet the 1e-9 parity bar and is off by
 * default.  nat <= 2 only (the generic evaluator and the fused path ignore the switch).                              */
#define FP_PREC_FP64  0
#define FP_PREC_MIXED 1
int fp_set_precision(fp_ctx *ctx, int mode);
int fp_get_precision(const fp_ctx *ctx);

/* Self-check of the FP32 pre-filter (DESIGN.md §5.2 claims it admits a superset of the candidates the pinned FP64 window
 * decision of PAPER.md:163,293 allows, so that counts and rates never depend on it).  fp_set_prefilter(ctx, 0) disables
 * every FP32 test -- each candidate then takes the pinned FP64 decision, 10-50x slower -- and fp_set_prefilter(ctx, 1)
 * restores the constants fp_setup derived.  Counts must be bit-identical either way (tests/test_gpu_fullsize.py).
 * Returns FP_OK or FP_EINVAL (null ctx).                                                                              */
int fp_set_prefilter(fp_ctx *ctx, int on);

/* Profiling of the library's own kernels (off by default; adds two cudaEventRecord per launch).                     */
int fp_profile_enable(fp_ctx *ctx, int on);
int fp_profile_reset(fp_ctx *ctx);
int fp_profile_get(fp_ctx *ctx, fp_profile *out);           /* synchronises the recorded events                      */

/* Pure-DFMA microbenchmark on all SMs: measured FP64 throughput of this device in TFLOP/s (roofline denominator
 * cross-check).                                                                                       */
int fp_probe_fp64_tflops(void *stream, double *tflops);

/* FP64 tensor-core microbenchmark (the dense-recast decision is taken by measurement, north_star
 * "only if ncu shows the gain"): mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4) on all SMs, 8 independent accumulator tiles per
 * warp.  out (HOST, 3 doubles), TFLOP/s: [0] DMMA alone, [1] DFMA alone in the same kernel shape (64 chains per thread),
 * [2] both kinds interleaved (flops of both / time: the sum of [0] and [1] if the two kinds issue side by side, their
 * harmonic combination if they share a pipe).                                                                        */
int fp_probe_dmma_tflops(void *stream, double out[3]);

/* Unit constants as derived inside the library from CODATA 2018: out[0]=C3, out[1]=C4 (1/ps), out[2]=C_kappa,
 * out[3]=hbar/kB (ps K).                                                                                              */
void fp_constants(double out[4]);

const char *fp_last_error(const fp_ctx *ctx);
const char *fp_version(void);
int fp_destroy(fp_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* FOURPHONON_H */
