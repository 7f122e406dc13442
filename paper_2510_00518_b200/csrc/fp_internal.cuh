// fp_internal.cuh -- shared declarations of the CUDA path (not part of the public ABI; see include/fourphonon.h).
//
// Notation follows SURVEY.md §8: lambda=(q,j) target, "row" = everything that is fixed while the last two legs vary:
//   3ph row = (target, channel)            free legs A = lambda'  (q',  j'),  B = lambda''  (q''  = q + s2 q')
//   4ph row = (target, channel, lambda')   free legs A = lambda'' (q'', j''), B = lambda''' (q''' = qbase + s2 q'')
// A candidate inside a row is the code  (qx*nb + ja)*nb + jb  with qx the free q-point of leg A.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>
#include <string>
#include <vector>

#include "../../include/fourphonon.h"

#define FP_MAX_NB 64          // branch-mask width of the enumerator (natoms <= 21)
#define FP_MAX_L 4096         // lcm of the mesh dimensions (1-D phase table in shared memory)

// One mode record, 32 B: the enumerator and the weight code read omega and v_g together.
struct __align__(32) ModeRec { double omega, vx, vy, vz; };

// Device-resident tables, passed to kernels by value.
struct FpDev {
    int nat, nb, N, N1, N2, N3;
    int L, m1, m2, m3;            // L = lcm(N1,N2,N3); m_mu = L/N_mu ; phase(q,R) = ph1d[(sum_mu i_mu m_mu n_mu) mod L]
    int Lmask;                    // L-1 if L is a power of two, else -1
    unsigned Lmagic;              // ceil(2^32 / L): x mod L by a multiply (phase_idx), L not a power of two
    double B[9];                  // B_mu = b_mu/N_mu, pinned arithmetic
    double scale, ncut, sigma_const, T;
    float pfK1, pfC2;             // FP32 pre-filter, stage 2: admit iff Delta_f^2 <= pfK1*|u_a-u_b|_f^2 + pfC2
    double pfCs, pfSlack;         // stage 1 table constants: n' = cs*|u|*(1+1e-6) + slack (k_tables)
    float pfNmax;                 // max n' over all modes; wmin/wmax: range of the non-zero frequencies (row_is_empty)
    double wmin, wmax;
    const ModeRec *rec;           // N*nb
    const float4 *recf;           // N*nb  {omega, B1.v, B2.v, B3.v} rounded to FP32; omega = NaN marks a zero mode
    const float2 *recn;           // nb*N, branch-major [j][iq]: {omega (NaN for zero modes), n'}; stage 1 admits iff
                                  // |Delta_f| <= n'_a + n'_b
    const double *occ;            // N*nb  f_lambda = 1/expm1(hbar omega/kB T)
    const double2 *evec;          // N*nb*nb mass-scaled eigenvectors e~ = e/sqrt(m)
    const double2 *evecc;         // N*nb*nb conj(e~): the conjugations of step 6 are table choices, not arithmetic
    const float2 *evec32, *evecc32;   // the same rounded to FP32 (mixed-precision evaluator, fp_set_precision)
    const double2 *ph1d;          // L
    const int *qc;                // N packed mesh coordinates i1 | i2<<10 | i3<<20   (N_mu <= 1024)
    const float2 *qmm;            // N  {min, max} of the non-zero frequencies of a q-point, rounded outward to FP32
    float pfW;                    // no pair of a q_A, q_B can pass stage 1 unless [Delta_min, Delta_max] meets [-pfW, pfW]
    // group path (fp_group.cu): one FP32 interval test per (A, B) pair, then the pinned decision
    const double2 *aux;           // N*nb  {f_lambda, 1/omega_lambda} (0, 0 for zero modes): the weight reads both together
    float gfC, gfD;               // window half-width bound of a pair: bnd = gfC * |u_a - u_b|_f + gfD
    float gfW;                    // upper bound of bnd over all pairs (tile vote)
    double thrC, invC;            // ncut*scale/sqrt(6) and sqrt(6)/scale: fast path of the decision and 1/sigma
    int pfOff;                    // fp_set_prefilter(ctx, 0): the stage-1 table of the fused kernel reads as n' = inf
};

// Anharmonic list in device layout: clusters sorted by contraction block.
//  ORDER 3: block = (atom j, atom k, Rj-Rk);  cl_meta0 = {i, Rk}            (phase conj(phi(q,Rk)) at level 0)
//  ORDER 4: block = (atom k, atom l, Rk-Rl);  cl_meta0 = {i, Rl}, cl_meta1 = {j, Rj-Rl}  (level 1)
// All cell offsets are stored reduced to [0,N_mu).
struct IfcDev {
    int n, nblk, ncomp;           // clusters, blocks, 27 or 81
    const int4 *cl_meta0;         // n
    const int4 *cl_meta1;         // n (ORDER 4 only)
    const double *phi;            // n*ncomp, block-sorted
    const int *blk_start;         // nblk+1 (CSR over clusters)
    const int4 *blk_meta;         // nblk {atomA | atomB<<16, d1, d2, d3}
    const int *seg;               // nat*nat+1 : block ranges per (atomA, atomB), blocks sorted by (atomA, atomB)
};

struct RowArgs {
    const int32_t *targets;       // device
    int64_t row0;                 // first row handled by this launch
    int qp_begin, nqp;            // 4ph only
    unsigned long long *prefiltered;   // nullable: += candidates admitted by the FP32 pre-filter (profiling)
    unsigned long long *evaluated;     // nullable: += list entries written by k_enum = matrix elements k_eval evaluates
    int sym;                      // 1: rows whose two free legs are both conjugated (3ph -, 4ph +- and --) list each
                                  // unordered pair of them once
    unsigned int *overflow;       // split path: += 1 for every (row, warp) list slot that filled up (the driver then
                                  // re-runs those rows through the fused kernel)
    int mglobal;                  // 3ph only: the block table Mhat of a row is read from the level-0 table in global memory
                                  // instead of a shared-memory copy (IFC3 lists too long for shared memory, ifc_mglobal())
};

// Group path: the targets of a super-chunk that share their q-point form a group; the rows of a group CTA -- 3ph:
// (member, channel); 4ph: (member, channel, q', j') for all j' -- share q_base, hence the momentum map q_A -> q_B and
// every record the enumerator loads, and differ only in their base energy.
struct GroupArgs {
    const int32_t *targets;       // device: the super-chunk's targets (local index t)
    const int4 *gdesc;            // ng     {q-point, first member (offset into gmem), members, j'_0 | n_j' << 16}: the rows of
                                  //        a 4ph group are (member, j') for j' in [j'_0, j'_0 + n_j')
    const int32_t *gmem;          // local target indices, grouped
    int ng, rmaxg;                // groups; largest row count of a group (stride of the list slots)
    int nu;                       // enumeration units per group CTA = list slots per row (enum_units())
    int qp_begin, nqp;            // 4ph only
    int64_t gid0;                 // first group CTA ((g, ch) for 3ph, (g, ch, q') for 4ph) of this launch
    int sym;                      // pair symmetry, as RowArgs::sym
    unsigned long long *prefiltered, *evaluated;   // nullable statistics (see RowArgs)
    unsigned int *overflow;
};

// One allowed process of a row in the split path: both free legs and the row-independent part of its weight.
struct __align__(16) ListEnt { uint32_t x, y; double w; };   // x = qA << 6 | jA (bit 31: both orderings of the pair passed),  y = qB << 6 | jB

struct EventRec { int cat; cudaEvent_t a, b; };

struct fp_ctx {
    FpDev d;
    IfcDev i3, i4;
    bool has3 = false, has4 = false;
    double vol = 0;               // |a1.(a2 x a3)|
    char *ws = nullptr;           // caller workspace
    size_t ws_bytes = 0, resident = 0;   // resident tables occupy [0, resident)
    int sm_count = 148;
    bool profiling = false;
    int path = FP_PATH_AUTO;      // fp_set_path
    bool sym34 = false, sym23 = false;   // IFC4 / IFC3 is symmetric under the exchange of its last two legs (fp_setup)
    bool use_sym = true;          // fp_set_symmetry
    int precision = FP_PREC_FP64; // fp_set_precision
    // time reversal (fp_set_target_symmetry): the mode arrays satisfy omega(-q,j) = omega(q,j), v(-q,j) = -v(q,j),
    // e(-q,j) = conj(e(q,j)) bit for bit (checked by fp_setup), so targets (q,j) and (-q,j) have the same rates and the
    // driver evaluates one of each pair (targets only in the irreducible part, N_list)
    bool trs_ok = false, use_trs = true;
    std::vector<int32_t> qpartner;   // N: index of -q
    bool pf_saved = false;        // fp_set_prefilter(ctx, 0) is in effect; the constants of fp_setup are kept here:
    float sv_pfK1 = 0, sv_pfC2 = 0, sv_pfNmax = 0, sv_pfW = 0, sv_gfC = 0, sv_gfD = 0, sv_gfW = 0;
    cudaStream_t side = nullptr;  // second stream of the split path: the enumerator of chunk k+1 runs beside the
    cudaEvent_t ev_enum[2] = {nullptr, nullptr}, ev_eval[2] = {nullptr, nullptr};   // evaluator of chunk k
    std::vector<EventRec> events;
    std::vector<cudaEvent_t> pool;   // profiling events recycled by fp_profile_reset
    fp_profile prof{};
    std::string err;
    int device = 0;               // the device fp_setup ran on
    double flops_elem3 = 0, flops_elem4 = 0;   // executed FP64 flops per matrix element of the evaluator (profile model)
};

enum { CAT_PRE = 0, CAT_RATES, CAT_REDUCE, CAT_ENUM, CAT_N };

// ---- kernel launchers (fp_kernels.cu) --------------------------------------------------------------------------------
void launch_tables(const FpDev &d, const double *omega, const double *eig, const double *vg, const double *masses_dev,
                   double hbar_over_kb, ModeRec *rec, float4 *recf, float2 *recn, double *occ, double2 *aux, double2 *evec, double2 *evecc, double2 *ph1d, int *qc,
                   float2 *qmm, unsigned long long *maxima /*2: bits of max omega, max |B v|_2*/, cudaStream_t st);
// fused rate kernel (fp_rates.cu)
void launch_pre3(const FpDev &d, const IfcDev &f, const int32_t *targets, int64_t nt, double2 *mhat, cudaStream_t st);
void launch_pre4(const FpDev &d, const IfcDev &f, const int32_t *targets, int64_t nt, double2 *t0, cudaStream_t st);
// only_flagged: redo pass of the split path -- only rows with counts[r] == 0xffffffff (a list slot filled up) are computed
cudaError_t launch_rates(int order, const FpDev &d, const IfcDev &f, const RowArgs &ra, int64_t nrows, const double2 *pre,
                         double2 *partial, uint32_t *counts, bool only_flagged, cudaStream_t st);
size_t rates_smem_bytes(const FpDev &d, const IfcDev &f, bool mglobal = false);
// true if the per-row table of an IFC3 list does not fit the shared memory of one SM: the 3ph kernels then read Mhat from
// global memory (L1/L2) -- slower per block, but the list length is no longer capped by it (include/fourphonon.h, Limits)
bool ifc_mglobal(const FpDev &d, const IfcDev &f, int order);
// per-process terms of explicit lists (fp_terms3 / fp_terms4): row r of the launch is ra.row0 + blockIdx.x
cudaError_t launch_terms(int order, const FpDev &d, const IfcDev &f, const RowArgs &ra, int64_t nrows, const double2 *pre,
                         const int64_t *offsets, int64_t list_base, const uint32_t *list, double scale, double *gamma_p,
                         cudaStream_t st);
// group path (fp_group.cu): group enumerator -> per-row process lists in the scratch -> tile evaluator
#define FP_GROUP_RMAX 64          // rows of one enumerator group (they share the scan of the two free legs)
int64_t enum_slot_entries(const FpDev &d);        // entries of one (row, warp) list slot that can never overflow
int enum_units(const FpDev &d);                   // enumeration units per group CTA = list slots per row
size_t eval_smem_bytes(const FpDev &d, const IfcDev &f, int ge, bool mglobal = false);   // dynamic shared memory of an evaluator tile of ge rows
// wcnt[(group CTA * rmaxg + row-in-group) * units + unit] = list entries written (0xffffffff: the slot filled up);
// work: a device counter the launcher zeroes (the units are dealt to the warps of a persistent grid)
cudaError_t launch_enum_g(int order, const FpDev &d, const GroupArgs &ga, int64_t ngc, int64_t capw, ListEnt *lists,
                          uint32_t *wcnt, unsigned int *work, int sm_count, cudaStream_t st);
// mixed: level-2 contraction in FP32 (nat <= 2 only; the generic evaluator stays FP64)
cudaError_t launch_eval_g(int order, const FpDev &d, const IfcDev &f, const GroupArgs &ga, int64_t ngc, const double2 *pre,
                          int64_t capw, const ListEnt *lists, const uint32_t *wcnt, int ge, double2 *partial,
                          uint32_t *counts, bool mixed, bool mglobal, cudaStream_t st);
void launch_finalize(int order, const FpDev &d, int64_t nt, int64_t rows_per_unit, const double2 *partial,
                     const uint32_t *counts, double c_over_n, double *gamma, double *wp, int64_t *cnt, cudaStream_t st);
void launch_kappa(const FpDev &d, const double *gamma_total, double pref, double *kappa, cudaStream_t st);
// process-list export (debug entry points fp_list3 / fp_list4): count -> scan -> ordered fill -> decode
void launch_count(int order, const FpDev &d, const RowArgs &ra, int64_t nrows, uint32_t *counts, cudaStream_t st);
void launch_scan(const uint32_t *counts, int64_t n, int64_t *offsets /*n+1*/, int64_t *block_sums, cudaStream_t st);
void launch_fill(int order, const FpDev &d, const RowArgs &ra, int64_t nrows, const int64_t *offsets, int64_t list_base,
                 uint32_t *list, cudaStream_t st);
void launch_decode(int order, const FpDev &d, const RowArgs &ra, const uint32_t *list, int64_t n, int32_t *out,
                   cudaStream_t st);
double run_fp64_probe(cudaStream_t st, int sm_count);
void run_dmma_probe(cudaStream_t st, int sm_count, double out[3]);

// Dynamic shared memory above 48 KB needs an opt-in per kernel AND per device (the attribute is a per-device setting):
// the granted size is cached per (kernel instantiation, device), under a lock.
struct SmemGrant { std::mutex mu; size_t granted[64] = {}; };
template <typename K>
static inline cudaError_t opt_in_smem(K kernel, size_t smem, SmemGrant &g) {   // opt-in limit is 227 KB minus the static part
    if (smem <= 48 * 1024) return cudaSuccess;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(g.mu);
    if (dev < 0 || dev >= 64 || smem > g.granted[dev]) {
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) g.granted[dev] = smem;
    }
    return cudaSuccess;
}
