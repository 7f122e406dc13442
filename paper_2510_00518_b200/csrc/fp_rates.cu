// fp_rates.cu -- the rate kernels of the FourPhonon hot path (SURVEY.md §8(a) rows a2/a3 + a5/a6 + a7) and the
// per-target pre-contraction.
//
//   k_pre3/k_pre4  per-target level-0 contraction of the IFC list with the target eigenvector
//   split path (default): Algorithm 3 -> Algorithm 4 of the paper, both on the device
//     k_enum       one CTA per row (3ph: (target, channel); 4ph: (target, channel, lambda')).  Each warp enumerates its
//                  share of the row's candidates (momentum modulo the mesh PAPER.md:155,288), filters them with the
//                  two-stage FP32 pre-filter, takes the window decision in the pinned FP64 arithmetic
//                  of SURVEY.md §8(c) step 3, computes the row-independent part of the weight and
//                  ballot-compacts the allowed processes into its list slot (16 bytes per process)
//     k_eval       one CTA per row: matrix element of every listed process (compute_Vp), two processes
//                  per lane against one pass over the row's contraction blocks, accumulation
//   fused path (small scratch, or a list slot that filled up)
//     k_rates      one CTA per row does all of the above; the process lists live and die in shared memory
//
// The window is decided twice.  A cheap FP32 pre-filter (tables recn / recf: omega and u = B v rounded to FP32) admits a
// proven superset of the allowed candidates (error budget in DESIGN.md §5.2, constants pfK1/pfC2 from fp_setup); only
// the ~2.5 % survivors pay for the pinned FP64 decision, which alone determines counts and rates.
//
// Contraction algebra: with the momentum modulo, phi(-q_last,R) factorises, so per row
//   V = sum_b phi(s2 qx, dR_b) sum_{xy} Mhat_b[x][y] A(atomA_b,x) conj(e~_B(atomB_b,y)),
// where the blocks b=(atomA,atomB,dR) merge all clusters that differ only in legs already fixed by the row, and
// Mhat_b folds the IFC values with the fixed legs' eigenvectors and phases.  A = e~_A (s2=+) or conj(e~_A) (s2=-).
#include <mutex>

#include "fp_device.cuh"

namespace {

// ---------------------------------------------------------------------------------------------------------------------
// a5 / a6 level 0: fold the target eigenvector (and the phase of the last leg at the target q) into the IFC list
// ---------------------------------------------------------------------------------------------------------------------
// 3ph: Mhat[t][b][x][y] = sum_{trip in b} conj(phi(q,Rk)) sum_a Phi^{a x y} e~_lam(i,a)          (x: leg j, y: leg k)
__global__ void __launch_bounds__(256) k_pre3(FpDev d, IfcDev f, const int32_t *targets, double2 *mhat) {
    int64_t t = blockIdx.x;
    int lam = targets[t];
    const double2 *e0 = d.evec + (size_t)lam * d.nb;
    int3 qm = premul(d, unpack_qc(d.qc[lam / d.nb]));
    for (int o = threadIdx.x; o < f.nblk * 9; o += blockDim.x) {
        int b = o / 9, xy = o - 9 * b;
        double2 acc = make_double2(0.0, 0.0);
        for (int c = f.blk_start[b]; c < f.blk_start[b + 1]; c++) {
            int4 m0 = f.cl_meta0[c];
            double2 ph = d.ph1d[phase_idx(d, qm, m0.y, m0.z, m0.w)];
            ph.y = -ph.y;                                             // phi(-q, Rk)
            const double *P = f.phi + (size_t)c * 27 + xy;
            double2 s = make_double2(0.0, 0.0);
            for (int a = 0; a < 3; a++) {
                double2 e = __ldg(e0 + 3 * m0.x + a);
                double v = P[9 * a];
                s.x = fma(v, e.x, s.x); s.y = fma(v, e.y, s.y);
            }
            cfma(acc, s, ph);
        }
        mhat[((size_t)t * f.nblk) * 9 + o] = acc;
    }
}
// 4ph: T0[t][c][b x y] = conj(phi(q,Rl)) sum_a Phi^{a b x y} e~_lam(i,a)
__global__ void __launch_bounds__(256) k_pre4(FpDev d, IfcDev f, const int32_t *targets, double2 *t0) {
    int64_t t = blockIdx.x;
    int lam = targets[t];
    const double2 *e0 = d.evec + (size_t)lam * d.nb;
    int3 qm = premul(d, unpack_qc(d.qc[lam / d.nb]));
    for (int o = threadIdx.x; o < f.n * 27; o += blockDim.x) {
        int c = o / 27, bxy = o - 27 * c;
        int4 m0 = f.cl_meta0[c];
        double2 ph = d.ph1d[phase_idx(d, qm, m0.y, m0.z, m0.w)];
        ph.y = -ph.y;
        const double *P = f.phi + (size_t)c * 81 + bxy;
        double2 s = make_double2(0.0, 0.0);
        for (int a = 0; a < 3; a++) {
            double2 e = __ldg(e0 + 3 * m0.x + a);
            double v = P[27 * a];
            s.x = fma(v, e.x, s.x); s.y = fma(v, e.y, s.y);
        }
        t0[(size_t)t * f.n * 27 + o] = cmul(s, ph);
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// a5 / a6 / a7: contraction + weights
// ---------------------------------------------------------------------------------------------------------------------
struct BlkSmem {
    double2 *M;        // nblk*9   Mhat_b[x][y]
    int4 *meta;        // nblk     {atomA | atomB<<16, d1, d2, d3}
    double2 *ph;       // L
    int *seg;          // nat*nat+1
};

// One block: u = sum_y (sum_x M[x][y] A[x]) Bc[y];  V += u * phase          (13 complex MAC = 52 DFMA)
__device__ __forceinline__ void block_term(const double2 *M, const double2 *A, const double2 *Bc, double2 ph, double2 &V) {
    double2 u = make_double2(0.0, 0.0);
#pragma unroll
    for (int y = 0; y < 3; y++) {
        double2 t = make_double2(0.0, 0.0);
#pragma unroll
        for (int x = 0; x < 3; x++) cfma(t, M[3 * x + y], A[x]);
        cfma(u, t, Bc[y]);
    }
    cfma(V, u, ph);
}

// NAT > 0: eigenvectors of both free legs live in registers, block loop statically split by (atomA, atomB).
// NAT == 0: generic atom count, eigenvector components are fetched per block (L1/L2-resident table).
// eA points at e~_A (s2=+) or conj(e~_A) (s2=-), eB at conj(e~_B); bs.ph holds phi (s2=+) or conj(phi) (s2=-): the
// conjugations of step 6 are table choices made once per row, not arithmetic in the loop.
template <int NAT>
__device__ __forceinline__ double2 contract_process(const FpDev &d, const BlkSmem &bs, const double2 *__restrict__ eA,
                                                    const double2 *__restrict__ eB, const double2 *A, const double2 *Bc,
                                                    int3 qmx) {
    double2 V = make_double2(0.0, 0.0);
    if constexpr (NAT > 0) {                                         // A, Bc: registers, loaded by the caller
#pragma unroll
        for (int a = 0; a < NAT; a++)
#pragma unroll
            for (int c = 0; c < NAT; c++) {
                const int b1 = bs.seg[a * NAT + c + 1];
                for (int b = bs.seg[a * NAT + c]; b < b1; b++) {
                    const int4 m = bs.meta[b];
                    block_term(bs.M + 9 * b, A + 3 * a, Bc + 3 * c, bs.ph[phase_idx(d, qmx, m.y, m.z, m.w)], V);
                }
            }
    } else {
        const int nat = d.nat;
        for (int a = 0; a < nat; a++) {                              // blocks are sorted by (atomA, atomB): one
            double2 Ag[3];                                           // eigenvector fetch per group, not per block
#pragma unroll
            for (int x = 0; x < 3; x++) Ag[x] = __ldg(eA + 3 * a + x);
            for (int c = 0; c < nat; c++) {
                const int b0 = bs.seg[a * nat + c], b1 = bs.seg[a * nat + c + 1];
                if (b0 == b1) continue;
                double2 Bg[3];
#pragma unroll
                for (int x = 0; x < 3; x++) Bg[x] = __ldg(eB + 3 * c + x);
                for (int b = b0; b < b1; b++) {
                    const int4 m = bs.meta[b];
                    block_term(bs.M + 9 * b, Ag, Bg, bs.ph[phase_idx(d, qmx, m.y, m.z, m.w)], V);
                }
            }
        }
    }
    return V;
}


// Two processes per lane against one pass over the row's blocks: every Mhat_b read from shared memory feeds 2 x 13
// complex MACs, and the two dependency chains interleave (NAT > 0 only).
template <int NAT>
__device__ __forceinline__ void contract_process2(const FpDev &d, const BlkSmem &bs, const double2 *A0, const double2 *B0,
                                                  int3 q0, const double2 *A1, const double2 *B1, int3 q1, double2 &V0,
                                                  double2 &V1) {
    V0 = make_double2(0.0, 0.0); V1 = make_double2(0.0, 0.0);
#pragma unroll
    for (int a = 0; a < NAT; a++)
#pragma unroll
        for (int c = 0; c < NAT; c++) {
            const int b1 = bs.seg[a * NAT + c + 1];
            for (int b = bs.seg[a * NAT + c]; b < b1; b++) {
                const int4 m = bs.meta[b];
                const double2 p0 = bs.ph[phase_idx(d, q0, m.y, m.z, m.w)], p1 = bs.ph[phase_idx(d, q1, m.y, m.z, m.w)];
                const double2 *M = bs.M + 9 * b;
                double2 u0 = make_double2(0.0, 0.0), u1 = make_double2(0.0, 0.0);
#pragma unroll
                for (int y = 0; y < 3; y++) {
                    double2 t0 = make_double2(0.0, 0.0), t1 = make_double2(0.0, 0.0);
#pragma unroll
                    for (int x = 0; x < 3; x++) {
                        const double2 mm = M[3 * x + y];
                        cfma(t0, mm, A0[3 * a + x]); cfma(t1, mm, A1[3 * a + x]);
                    }
                    cfma(u0, t0, B0[3 * c + y]); cfma(u1, t1, B1[3 * c + y]);
                }
                cfma(V0, u0, p0); cfma(V1, u1, p1);
            }
        }
}

// The same for any atom count: eigenvector components are fetched per atom group (A once per atomA, B once per
// (atomA, atomB) pair with blocks), every Mhat_b read feeds both processes.
__device__ __forceinline__ void contract_process2_generic(const FpDev &d, const BlkSmem &bs, const double2 *__restrict__ eA0,
                                                          const double2 *__restrict__ eB0, int3 q0,
                                                          const double2 *__restrict__ eA1, const double2 *__restrict__ eB1,
                                                          int3 q1, double2 &V0, double2 &V1) {
    V0 = make_double2(0.0, 0.0); V1 = make_double2(0.0, 0.0);
    const int nat = d.nat;
    for (int a = 0; a < nat; a++) {
        if (bs.seg[a * nat] == bs.seg[(a + 1) * nat]) continue;
        double2 A0[3], A1[3];
#pragma unroll
        for (int x = 0; x < 3; x++) { A0[x] = __ldg(eA0 + 3 * a + x); A1[x] = __ldg(eA1 + 3 * a + x); }
        for (int c = 0; c < nat; c++) {
            const int b0 = bs.seg[a * nat + c], b1 = bs.seg[a * nat + c + 1];
            if (b0 == b1) continue;
            double2 B0[3], B1[3];
#pragma unroll
            for (int y = 0; y < 3; y++) { B0[y] = __ldg(eB0 + 3 * c + y); B1[y] = __ldg(eB1 + 3 * c + y); }
            for (int b = b0; b < b1; b++) {
                const int4 m = bs.meta[b];
                const double2 p0 = bs.ph[phase_idx(d, q0, m.y, m.z, m.w)], p1 = bs.ph[phase_idx(d, q1, m.y, m.z, m.w)];
                const double2 *M = bs.M + 9 * b;
                double2 u0 = make_double2(0.0, 0.0), u1 = make_double2(0.0, 0.0);
#pragma unroll
                for (int y = 0; y < 3; y++) {
                    double2 t0 = make_double2(0.0, 0.0), t1 = make_double2(0.0, 0.0);
#pragma unroll
                    for (int x = 0; x < 3; x++) {
                        const double2 mm = M[3 * x + y];
                        cfma(t0, mm, A0[x]); cfma(t1, mm, A1[x]);
                    }
                    cfma(u0, t0, B0[y]); cfma(u1, t1, B1[y]);
                }
                cfma(V0, u0, p0); cfma(V1, u1, p1);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// a2/a3 + a5/a6 + a7: fused enumerate -> shared-memory queue -> evaluate
// ---------------------------------------------------------------------------------------------------------------------
constexpr int RATES_MINB = 4;                 // k_rates: 128 registers
constexpr int RT = 128;                       // threads per row CTA
constexpr int RW = RT / 32;                   // warps
constexpr int EVT = 128;                      // threads of a k_eval CTA (measured on B200, config 3: 32 -> 1363 ms, 64 -> 1232,
                                              // 128 -> 1138, 256 -> 1425 per step: the row set-up wants several warps)
constexpr int PCAP = 32 + 32 * 36;            // pending queue: < 32 left over + one 6x6 sub-tile of 32 q-points
constexpr int QCAP = 64;                      // evaluation queue: < 32 left over + one stage-2 round

// Evaluation-queue entry: {qA << 6 | jA, qB << 6 | jB}: both legs are addressable at once, so every load of a batch
// is issued before the first dependent instruction.
// Pending-queue entry: qx << 12 | ja << 6 | jb   (N <= 2^20 q-points, nb <= 64)
__device__ __forceinline__ uint32_t pack_code(int qx, int ja, int jb) { return ((uint32_t)qx << 12) | (ja << 6) | jb; }

struct RowWeights {
    double wrow;        // omega (3ph) or omega * omega' (4ph)
    double occ_row;     // 1 (3ph) or (1+f') | f' divided by f (4ph)
};

template <int ORDER, int NAT>
__device__ __forceinline__ void eval_process(const FpDev &d, const BlkSmem &bs, const Row &row,
                                             const RowWeights &rw, uint2 ent, bool active, double &sG, double &sW,
                                             unsigned &cnt) {
    const int qx = (int)(ent.x >> 6);
    const int p = qx * d.nb + (int)(ent.x & 63u), lamB = (int)(ent.y >> 6) * d.nb + (int)(ent.y & 63u);
    // all loads of the batch up front: mode records, occupations, mesh coordinates, both eigenvectors
    const double2 *eA = (row.s2 > 0 ? d.evec : d.evecc) + (size_t)p * d.nb, *eB = d.evecc + (size_t)lamB * d.nb;
    const ModeRec a = load_rec(d.rec + p), b = load_rec(d.rec + lamB);
    const double fa = __ldg(d.occ + p), fb = __ldg(d.occ + lamB);
    const int3 xc = unpack_qc(__ldg(d.qc + qx));
    double2 A[3 * (NAT > 0 ? NAT : 1)], Bc[3 * (NAT > 0 ? NAT : 1)];
    if constexpr (NAT > 0) {
        load_evec<3 * NAT>(eA, A);
        load_evec<3 * NAT>(eB, Bc);
    }
    // the decision, in the pinned arithmetic
    const double sig = sigma_pinned(d, a, b);
    const double delta = __dsub_rn(row.s2 > 0 ? __dadd_rn(row.Obase, a.omega) : __dsub_rn(row.Obase, a.omega), b.omega);
    const bool ok = active && a.omega != 0.0 && b.omega != 0.0 && sig > 0.0 && fabs(delta) <= __dmul_rn(d.ncut, sig);
    if (!__any_sync(0xffffffffu, ok)) return;
    const double2 V = contract_process<NAT>(d, bs, eA, eB, A, Bc, premul(d, xc));
    const double v2 = V.x * V.x + V.y * V.y;
    // weights: g = exp(-(Delta/sigma)^2)/(sigma sqrt(pi)), WP = occ * g / (omega omega' omega'' [omega'''])
    const double W = rw.wrow * a.omega * b.omega;
    const double t = 1.0 / (sig * W);
    const double rr = delta * (t * W);
    const double g_over_W = exp(-(rr * rr)) * t * 0.56418958354775628695;       // 1/sqrt(pi)
    double occ;
    if (ORDER == 3) occ = row.s2 > 0 ? (fa - fb) : (fa + fb + 1.0);
    else occ = rw.occ_row * (row.s2 > 0 ? 1.0 + fa : fa) * fb;
    const double WP = occ * g_over_W;
    if (ok) {
        sW += WP;
        sG = fma(WP, v2, sG);
        cnt++;
    }
}

// FP32 pre-filter, stage 2, of one candidate code (table recf): Delta_f^2 <= K1 |u_a - u_b|_f^2 + C2
__device__ __forceinline__ bool prefilter2(const FpDev &d, const Row &row, float basef, uint32_t code, uint2 &ent) {
    const int qx = (int)(code >> 12), ja = (int)((code >> 6) & 63u), jb = (int)(code & 63u);
    const int ql = q_index(d, q_add(d, row.qb, row.s2, unpack_qc(__ldg(d.qc + qx))));
    ent = make_uint2(((uint32_t)qx << 6) | (uint32_t)ja, ((uint32_t)ql << 6) | (uint32_t)jb);   // evaluation-queue entry
    const float4 A = __ldg(d.recf + (size_t)qx * d.nb + ja), B = __ldg(d.recf + (size_t)ql * d.nb + jb);
    const float dl = (row.s2 > 0 ? basef + A.x : basef - A.x) - B.x;
    const float dx = A.y - B.y, dy = A.z - B.z, dz = A.w - B.w;
    const float s = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    return dl * dl <= fmaf(d.pfK1, s, d.pfC2);
}

// No candidate of the row can pass the window: |Delta| <= ncut sigma <= n_a + n_b <= 2 nmax for every allowed process,
// and Delta = base + s2 omega_A - omega_B with both legs' frequencies in [wmin, wmax] (the non-zero modes).
__device__ __forceinline__ bool row_is_empty(const FpDev &d, const Row &row) {
    const double w2 = 2.0 * (double)d.pfNmax, lo = d.wmin, hi = d.wmax;
    const double dmin = row.s2 > 0 ? row.Obase + lo - hi : row.Obase - 2.0 * hi;
    const double dmax = row.s2 > 0 ? row.Obase + hi - lo : row.Obase - 2.0 * lo;
    return dmin > w2 || dmax < -w2;
}

// Shared-memory tables of one row (layout mirrored by tables_smem_bytes()): Mhat, phases, level-1 eigenvector, block
// metadata, (atomA, atomB) segments.  Returns the first free byte after them.
template <int ORDER>
__device__ __forceinline__ unsigned char *setup_row_tables(const FpDev &d, const IfcDev &f, const Row &row,
                                                           const double2 *pre, unsigned char *smem_raw, BlkSmem &bs,
                                                           RowWeights &rw) {
    bs.M = reinterpret_cast<double2 *>(smem_raw);
    bs.ph = bs.M + 9 * f.nblk;
    double2 *e1 = bs.ph + d.L;                                        // nb entries (level 1 of ORDER 4)
    bs.meta = reinterpret_cast<int4 *>(e1 + d.nb);
    bs.seg = reinterpret_cast<int *>(bs.meta + f.nblk);
    for (int i = threadIdx.x; i < f.nblk; i += blockDim.x) bs.meta[i] = f.blk_meta[i];
    for (int i = threadIdx.x; i <= d.nat * d.nat; i += blockDim.x) bs.seg[i] = f.seg[i];
    if (ORDER == 3) {
        const double2 *src = pre + (size_t)row.t * f.nblk * 9;
        for (int i = threadIdx.x; i < f.nblk * 9; i += blockDim.x) bs.M[i] = src[i];
    } else {
        // level 1: Mhat_b[x][y] = sum_{c in b} phi(s1 q', Rj-Rl) sum_be T0[c][be][x][y] A'(j_c, be)
        for (int i = threadIdx.x; i < d.L; i += blockDim.x) {
            double2 p = d.ph1d[i];
            if (row.s1 < 0) p.y = -p.y;
            bs.ph[i] = p;
        }
        const double2 *ev1 = (row.s1 > 0 ? d.evec : d.evecc) + (size_t)row.lam1 * d.nb;
        for (int i = threadIdx.x; i < d.nb; i += blockDim.x) e1[i] = ev1[i];
        __syncthreads();
        const int3 qm1 = premul(d, unpack_qc(d.qc[row.lam1 / d.nb]));
        const double2 *T0 = pre + (size_t)row.t * f.n * 27;
        for (int o = threadIdx.x; o < f.nblk * 9; o += blockDim.x) {
            int b = o / 9, xy = o - 9 * b;
            double2 acc = make_double2(0.0, 0.0);
            for (int c = f.blk_start[b]; c < f.blk_start[b + 1]; c++) {
                int4 m1 = f.cl_meta1[c];
                double2 ph = bs.ph[phase_idx(d, qm1, m1.y, m1.z, m1.w)];
                double2 s = make_double2(0.0, 0.0);
#pragma unroll
                for (int be = 0; be < 3; be++) cfma(s, T0[(size_t)c * 27 + 9 * be + xy], e1[3 * m1.x + be]);
                cfma(acc, s, ph);
            }
            bs.M[o] = acc;
        }
        __syncthreads();
    }
    for (int i = threadIdx.x; i < d.L; i += blockDim.x) {                     // phases of the free legs: phi(s2 qx, dR)
        double2 p = d.ph1d[i];
        if (row.s2 < 0) p.y = -p.y;
        bs.ph[i] = p;
    }
    __syncthreads();
    rw.wrow = d.rec[row.lam].omega;
    rw.occ_row = 1.0;
    if (ORDER == 4) {
        const double f1 = d.occ[row.lam1];
        rw.wrow *= d.rec[row.lam1].omega;
        rw.occ_row = (row.s1 > 0 ? 1.0 + f1 : f1) / d.occ[row.lam];
    }
    return reinterpret_cast<unsigned char *>(bs.seg + ((d.nat * d.nat + 1 + 3) & ~3));
}

// FP32 pre-filter, stage 1, of one sub-tile (32 q-points x TILE x TILE branch pairs, table recn): each lane owns one
// q-point and admits a pair iff |Delta_f| <= n'_a + n'_b (sigma <= cs(|u_a| + |u_b|)); survivors are appended, in
// candidate order, to the warp's pending queue.  Returns the new queue length (warp-uniform).
template <int TILE>
__device__ __forceinline__ int stage1_step(const FpDev &d, const Row &row, float basef, int tile, int ja0, int jb0,
                                           int lane, uint32_t *pend, int wp, bool canonical_only = false) {
    const float fnan = __int_as_float(0x7fc00000);
    const int qx = (tile << 5) + lane;
    const bool inq = qx < d.N;
    const int qs = inq ? qx : 0;
    const int ql = q_index(d, q_add(d, row.qb, row.s2, unpack_qc(d.qc[qs])));
    // Tile test, one warp vote before the branch records are loaded: a q-point whose frequency ranges cannot bring Delta
    // into [-pfW, pfW] holds no stage-1 survivor (most tiles of the ++ and -- rows with a large base energy); with the
    // pair symmetry neither does one with q_A above q_B (on a mesh with N1 N2 >= 32 every tile whose i3 plane lies above
    // the plane of its q_B: half of the scan).
    {
        const float2 mA = __ldg(d.qmm + qs), mB = __ldg(d.qmm + ql);
        const float dmin = (row.s2 > 0 ? basef + mA.x : basef - mA.y) - mB.y;
        const float dmax = (row.s2 > 0 ? basef + mA.y : basef - mA.x) - mB.x;
        const bool live = inq && dmin <= d.pfW && dmax >= -d.pfW && (!canonical_only || qs <= ql);
        if (!__any_sync(0xffffffffu, live)) return wp;
    }
    const float2 *pa = d.recn + (size_t)ja0 * d.N + qs, *pb = d.recn + (size_t)jb0 * d.N + ql;   // branch-major table
    float lo[TILE], hi[TILE];
#pragma unroll
    for (int i = 0; i < TILE; i++) {
        const float2 A = __ldg(pa + (size_t)i * d.N);                 // omega_f = NaN for zero modes: never admitted
        const float ba = inq ? (row.s2 > 0 ? basef + A.x : basef - A.x) : fnan;
        lo[i] = ba - A.y; hi[i] = ba + A.y;
    }
    uint64_t mask = 0;
#pragma unroll
    for (int k = 0; k < TILE; k++) {
        const float2 B = __ldg(pb + (size_t)k * d.N);
        const float bl = B.x - B.y, bh = B.x + B.y;
#pragma unroll
        for (int i = 0; i < TILE; i++)
            if (bl <= hi[i] && bh >= lo[i]) mask |= 1ull << (8 * i + k);
    }
    if (canonical_only) {                                             // pair symmetry: keep mode A <= mode B only
        uint64_t upper = 0;                                           // bit 8 i + k with ja0 + i <= jb0 + k
#pragma unroll
        for (int i = 0; i < TILE; i++)
#pragma unroll
            for (int k = 0; k < TILE; k++)
                if (ja0 + i <= jb0 + k) upper |= 1ull << (8 * i + k);
        mask = qs < ql ? mask : qs == ql ? (mask & upper) : 0ull;
    }
    const unsigned c = __popcll(mask);                                // ordered append to the pending queue
    unsigned incl = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    unsigned pos = wp + incl - c;
    while (mask) {
        const int bit = __ffsll((long long)mask) - 1;
        mask &= mask - 1;
        pend[pos++] = pack_code(qx, ja0 + (bit >> 3), jb0 + (bit & 7));
    }
    return wp + (int)__shfl_sync(0xffffffffu, incl, 31);
}

// sub-tile decomposition of the enumeration: step -> (q-tile, ja0, jb0)
template <int TILE, bool ONE_SUB>
struct Steps {
    int nsub, nsteps;
    __device__ __forceinline__ Steps(const FpDev &d) {
        nsub = ONE_SUB ? 1 : d.nb / TILE;
        nsteps = ((d.N + 31) >> 5) * nsub * nsub;
    }
    __device__ __forceinline__ void decode(int step, int &tile, int &ja0, int &jb0) const {
        if (ONE_SUB) { tile = step; ja0 = 0; jb0 = 0; return; }
        tile = step / (nsub * nsub);
        const int sub = step - tile * nsub * nsub;
        ja0 = (sub / nsub) * TILE; jb0 = (sub - (sub / nsub) * nsub) * TILE;
    }
};

// ---------------------------------------------------------------------------------------------------------------------
// fused path: enumerate -> shared-memory queues -> evaluate, one CTA per row (used when the scratch is too small for
// process lists; the process lists of Algorithm 3, live and die in shared memory)
// ---------------------------------------------------------------------------------------------------------------------
template <int ORDER, int NAT, int TILE>
__global__ void __launch_bounds__(RT, RATES_MINB) k_rates(FpDev d, IfcDev f, RowArgs ra, const double2 *pre, double2 *partial,
                                                 uint32_t *counts, bool only_flagged) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double red[32];
    __shared__ unsigned redc[32];
    __shared__ int tailn[RW];
    const int64_t r = blockIdx.x;
    if (only_flagged && counts[r] != 0xffffffffu) return;             // redo pass: only rows whose list slot filled up
    const Row row = make_row<ORDER>(d, ra, ra.row0 + r);
    if (!row.valid || row_is_empty(d, row)) {                         // item 8: zero modes are never a leg
        if (threadIdx.x == 0) { partial[r] = make_double2(0.0, 0.0); counts[r] = 0; }
        return;
    }
    BlkSmem bs;
    RowWeights rw;
    uint2 *evq = reinterpret_cast<uint2 *>(setup_row_tables<ORDER>(d, f, row, pre, smem_raw, bs, rw));   // RW*QCAP
    uint2 *tailbuf = evq + RW * QCAP;                                                  // RW*32 (merged tails)
    uint32_t *pendq = reinterpret_cast<uint32_t *>(tailbuf + RW * 32);                // RW*PCAP

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t *pend = pendq + warp * PCAP;                             // stage-1 survivors of this warp
    uint2 *myq = evq + warp * QCAP;                                   // stage-2 survivors, evaluated 32 at a time
    int wp = 0, wq = 0;                                               // entries in pend / myq (warp-uniform)
    double sG = 0.0, sW = 0.0;
    unsigned cnt = 0, nadm = 0;

    // ---- one loop, one evaluation site: evaluate a full batch if one is queued, else refill the queue -------------------
    //   stage 1 (stage1_step) and stage 2 (prefilter2) admit every candidate the pinned FP64 decision allows
    //   (DESIGN.md §5.2), which alone decides.
    const float basef = (float)row.Obase;
    constexpr bool ONE_SUB = (NAT > 0 && 3 * NAT == TILE);            // nb == TILE: one sub-tile per q-tile
    const Steps<TILE, ONE_SUB> steps(d);
    int step = warp, phase = 0, tbase = 0, total = 0;                 // phase 0 enumerate, 1 flush pend, 2 merged tails
    for (;;) {
        __syncwarp();
        uint2 ent = make_uint2(0u, 0u);
        bool act = false, have = false;
        if (wq >= 32) {
            wq -= 32; ent = myq[wq + lane]; act = true; have = true;
        } else if (phase == 2) {
            if (tbase >= total) break;
            const int idx = tbase + lane;
            act = idx < total; ent = tailbuf[act ? idx : tbase]; tbase += RT; have = true;
        }
        if (have) {
            eval_process<ORDER, NAT>(d, bs, row, rw, ent, act, sG, sW, cnt);
            continue;
        }
        if (wp >= 32 || (phase == 1 && wp > 0)) {                     // stage 2 on up to 32 pending candidates
            const int n = wp < 32 ? wp : 32;
            wp -= n;
            const bool in = lane < n;
            const uint32_t c2 = pend[wp + (in ? lane : 0)];
            uint2 e2;
            const bool pass = prefilter2(d, row, basef, c2, e2) && in;
            const unsigned bal = __ballot_sync(0xffffffffu, pass);
            if (pass) myq[wq + __popc(bal & ((1u << lane) - 1u))] = e2;
            wq += __popc(bal);
            nadm += pass ? 1u : 0u;
            continue;
        }
        if (phase == 0) {
            if (step >= steps.nsteps) { phase = 1; continue; }
            int tile, ja0, jb0;
            steps.decode(step, tile, ja0, jb0);
            step += RW;
            wp = stage1_step<TILE>(d, row, basef, tile, ja0, jb0, lane, pend, wp);
            continue;
        }
        // phase 1 with pend empty and fewer than 32 queued: merge the leftovers of all warps so that at most one batch
        // of the row is partially filled
        if (lane == 0) tailn[warp] = wq;
        __syncthreads();
        int off = 0;
#pragma unroll
        for (int w = 0; w < RW; w++) {
            const int n = tailn[w];
            if (w < warp) off += n;
            total += n;
        }
        if (lane < wq) tailbuf[off + lane] = myq[lane];
        __syncthreads();
        wq = 0; phase = 2; tbase = warp * 32;
    }

    const double tG = block_sum<double>(sG, red);
    const double tW = block_sum<double>(sW, red);
    const unsigned tC = block_sum<unsigned>(cnt, redc);
    if (threadIdx.x == 0) { partial[r] = make_double2(tG, tW); counts[r] = tC; }
    if (ra.prefiltered) {                                             // profiling only: pre-filter survivors
        const unsigned tA = block_sum<unsigned>(nadm, redc);
        if (threadIdx.x == 0) atomicAdd(ra.prefiltered, (unsigned long long)tA);
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// split path (the default): process lists in HBM, Algorithm 3 -> Algorithm 4 of the paper with both
// halves on the device.  The enumerator needs ~40 registers and no FP64 pipe, the evaluator 128 registers and little
// else: as separate kernels each runs at its own occupancy, and (on two streams) the enumerator of the next chunk of
// rows fills the issue slots the FP64-bound evaluator leaves empty.
//
// List layout: every (row, warp) owns a slot of capw entries (capw = all candidates the warp can meet, so nothing can
// overflow; untouched slot space costs no traffic); wcnt[row*RW + warp] is the number of entries written.  Entry order
// inside a slot is the enumerator's (deterministic), so sums are reproducible run to run.
// ---------------------------------------------------------------------------------------------------------------------
static_assert(RW == 4, "k_eval reads the four warp counts of a row as one uint4");

// Enumerator: stage 1 and 2 of the FP32 pre-filter, then -- for the survivors only -- the pinned FP64 decision
// (SURVEY.md §8(c) step 3), which alone determines what is written, and the row-independent part of the
// weight (a7).  With ~48 registers per thread ten CTAs fit on an SM, which hides the gather latency of the decision.
template <int ORDER, int TILE, bool ONE_SUB>
__global__ void __launch_bounds__(RT, 8) k_enum(FpDev d, RowArgs ra, int64_t capw, ListEnt *lists, uint32_t *wcnt,
                                                uint32_t *pcnt) {
    __shared__ uint32_t pendq[RW * PCAP];
    const int64_t r = blockIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const Row row = make_row<ORDER>(d, ra, ra.row0 + r);
    unsigned nout = 0, nadm = 0, nproc = 0;
    bool ovf = false;                                                 // the slot filled up: the row is redone by k_rates
    // pair symmetry (fp_set_symmetry): in the 3ph - and the 4ph +- and -- channels (s2 < 0) the two free legs enter V and the
    // weight in the same way, so only mode A <= mode B is listed; its entry carries the weights of both orderings, each with its own
    // window decision in the pinned arithmetic
    const bool sym = ra.sym && row.s2 < 0;
    if (row.valid && !row_is_empty(d, row)) {                         // item 8: zero modes are never a leg
        ListEnt *out = lists + ((size_t)r * RW + warp) * (size_t)capw;
        uint32_t *pend = pendq + warp * PCAP;
        const float basef = (float)row.Obase;
        const Steps<TILE, ONE_SUB> steps(d);
        int wp = 0;
        for (int step = warp; step < steps.nsteps; step += RW) {
            int tile, ja0, jb0;
            steps.decode(step, tile, ja0, jb0);
            wp = stage1_step<TILE>(d, row, basef, tile, ja0, jb0, lane, pend, wp, sym);
            __syncwarp();
            const bool last = step + RW >= steps.nsteps;
            while (wp >= 32 || (last && wp > 0)) {                    // stage 2, 32 pending candidates at a time
                const int n = wp < 32 ? wp : 32;
                wp -= n;
                const bool in = lane < n;
                const uint32_t c2 = pend[wp + (in ? lane : 0)];
                // stage 2 and the loads of stage 3 are issued together (one L2 round trip instead of two; a quarter of the
                // FP64 records is fetched for candidates stage 2 then rejects)
                const int qx = (int)(c2 >> 12), ja = (int)((c2 >> 6) & 63u), jb = (int)(c2 & 63u);
                const int ql = q_index(d, q_add(d, row.qb, row.s2, unpack_qc(__ldg(d.qc + qx))));
                const int p = qx * d.nb + ja, lamB = ql * d.nb + jb;
                const uint2 e2 = make_uint2(((uint32_t)qx << 6) | (uint32_t)ja, ((uint32_t)ql << 6) | (uint32_t)jb);
                const float4 Af = __ldg(d.recf + p), Bf = __ldg(d.recf + lamB);
                const ModeRec a = load_rec(d.rec + p), b = load_rec(d.rec + lamB);
                const double fa = __ldg(d.occ + p), fb = __ldg(d.occ + lamB);
                const float dl = (row.s2 > 0 ? basef + Af.x : basef - Af.x) - Bf.x;
                const float dx = Af.y - Bf.y, dy = Af.z - Bf.z, dz = Af.w - Bf.w;
                const bool pass = in && dl * dl <= fmaf(d.pfK1, fmaf(dz, dz, fmaf(dy, dy, dx * dx)), d.pfC2);
                bool ok = false;
                double w = 0.0;
                if (pass) {                                           // stage 3: the decision, in the pinned arithmetic
                    const double sig = sigma_pinned(d, a, b);
                    const double delta = __dsub_rn(row.s2 > 0 ? __dadd_rn(row.Obase, a.omega) : __dsub_rn(row.Obase, a.omega), b.omega);
                    ok = a.omega != 0.0 && b.omega != 0.0 && sig > 0.0 && fabs(delta) <= __dmul_rn(d.ncut, sig);
                    // weight without the row factors: occ(f_A, f_B) g / (omega_A omega_B),  g = exp(-(Delta/sigma)^2)/(sigma sqrt(pi))
                    const double W = a.omega * b.omega;
                    const double t = 1.0 / (sig * W);
                    const double rr = delta * (t * W);
                    double occ;
                    if (ORDER == 3) occ = row.s2 > 0 ? (fa - fb) : (fa + fb + 1.0);   // symmetric in (A, B) for s2 < 0
                    else occ = (row.s2 > 0 ? 1.0 + fa : fa) * fb;
                    w = occ * (exp(-(rr * rr)) * t * 0.56418958354775628695);   // 1/sqrt(pi)
                    if (!ok) w = 0.0;
                    if (sym) {                                        // the other ordering: Delta' = (Obase - omega_B) - omega_A
                        const double delta2 = __dsub_rn(__dsub_rn(row.Obase, b.omega), a.omega);
                        const bool ok2 = p != lamB &&                 // (A = B is its own partner: one process; only a fixed sigma admits it)
                                         a.omega != 0.0 && b.omega != 0.0 && sig > 0.0 && fabs(delta2) <= __dmul_rn(d.ncut, sig);
                        if (ok2) {
                            const double r2 = delta2 * (t * W);
                            w += delta2 == delta ? occ * (exp(-(rr * rr)) * t * 0.56418958354775628695)
                                                 : occ * (exp(-(r2 * r2)) * t * 0.56418958354775628695);
                        }
                        nproc += (ok ? 1u : 0u) + (ok2 ? 1u : 0u);
                        ok = ok || ok2;
                    } else {
                        nproc += ok ? 1u : 0u;
                    }
                }
                const unsigned bal = __ballot_sync(0xffffffffu, ok);
                if (nout + __popc(bal) > (unsigned)capw) ovf = true;  // warp-uniform
                else {
                    if (ok) {
                        ListEnt e; e.x = e2.x; e.y = e2.y; e.w = w;
                        out[nout + __popc(bal & ((1u << lane) - 1u))] = e;
                    }
                    nout += __popc(bal);
                }
                nadm += pass ? 1u : 0u;
            }
            __syncwarp();
        }
    }
    for (int o = 16; o > 0; o >>= 1) nproc += __shfl_down_sync(0xffffffffu, nproc, o);
    if (lane == 0) {
        wcnt[r * RW + warp] = ovf ? 0xffffffffu : nout;
        pcnt[r * RW + warp] = nproc;
        if (ovf) atomicAdd(ra.overflow, 1u);
        else if (ra.evaluated && nout) atomicAdd(ra.evaluated, (unsigned long long)nout);
    }
    if (ra.prefiltered) {                                             // profiling only: pre-filter survivors
        for (int o = 16; o > 0; o >>= 1) nadm += __shfl_down_sync(0xffffffffu, nadm, o);
        if (lane == 0 && nadm) atomicAdd(ra.prefiltered, (unsigned long long)nadm);
    }
}

// Evaluator: |V|^2 of every listed process (level-2 contraction) and the row sums.  Every entry is an allowed process,
// so the row count is the list length; the row factors of the weight (1/omega[omega'], occupation of lambda') multiply
// the sums once.
// k_eval: two processes per lane, 168 registers, 3 CTAs per SM
template <int ORDER, int NAT>
__global__ void __launch_bounds__(EVT, 3 * (RT / EVT)) k_eval(FpDev d, IfcDev f, RowArgs ra, const double2 *pre, int64_t capw,
                                                      const ListEnt *lists, const uint32_t *wcnt, const uint32_t *pcnt,
                                                      double2 *partial, uint32_t *counts) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double red[32];
    const int64_t r = blockIdx.x;
    const uint4 wc = __ldg(reinterpret_cast<const uint4 *>(wcnt) + r);
    const bool ovf = (wc.x & wc.y & wc.z & wc.w) == 0xffffffffu || wc.x == 0xffffffffu || wc.y == 0xffffffffu ||
                     wc.z == 0xffffffffu || wc.w == 0xffffffffu;      // a slot of the row filled up: redone by k_rates
    const unsigned p1 = wc.x, p2 = p1 + wc.y, p3 = p2 + wc.z, total = ovf ? 0u : p3 + wc.w;
    if (total == 0) {                                                 // (0xffffffff marks the row for the redo pass)
        if (threadIdx.x == 0) { partial[r] = make_double2(0.0, 0.0); counts[r] = ovf ? 0xffffffffu : 0u; }
        return;
    }
    const Row row = make_row<ORDER>(d, ra, ra.row0 + r);
    BlkSmem bs;
    RowWeights rw;
    setup_row_tables<ORDER>(d, f, row, pre, smem_raw, bs, rw);

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const ListEnt *slot = lists + (size_t)r * RW * (size_t)capw;
    // the four slots of the row read as one list: entry i lives in slot w = #{k : i >= p_k} at offset i - p_w
    auto fetch = [&](unsigned i) -> ListEnt {
        const unsigned w = (i >= p1) + (i >= p2) + (i >= p3);
        const unsigned off = i - (w == 0 ? 0u : w == 1 ? p1 : w == 2 ? p2 : p3);
        const uint4 v = __ldg(reinterpret_cast<const uint4 *>(slot + (size_t)w * (size_t)capw + off));
        ListEnt e; e.x = v.x; e.y = v.y; e.w = __hiloint2double((int)v.w, (int)v.z);
        return e;
    };
    double sG = 0.0, sW = 0.0;
    for (unsigned base = warp * 64; base < total; base += 2 * EVT) {   // 64 processes per warp pass, two per lane
        const bool act0 = base + lane < total, act1 = base + 32 + lane < total;
        const ListEnt e0 = fetch(act0 ? base + lane : base), e1 = fetch(act1 ? base + 32 + lane : base);
        const int qx0 = (int)(e0.x >> 6), qx1 = (int)(e1.x >> 6);
        const double2 *eA0 = (row.s2 > 0 ? d.evec : d.evecc) + ((size_t)qx0 * d.nb + (e0.x & 63u)) * d.nb;
        const double2 *eA1 = (row.s2 > 0 ? d.evec : d.evecc) + ((size_t)qx1 * d.nb + (e1.x & 63u)) * d.nb;
        const double2 *eB0 = d.evecc + ((size_t)(e0.y >> 6) * d.nb + (e0.y & 63u)) * d.nb;
        const double2 *eB1 = d.evecc + ((size_t)(e1.y >> 6) * d.nb + (e1.y & 63u)) * d.nb;
        const int3 xc0 = unpack_qc(__ldg(d.qc + qx0)), xc1 = unpack_qc(__ldg(d.qc + qx1));
        double2 V0, V1;
        if constexpr (NAT > 0) {
            double2 A0[3 * (NAT > 0 ? NAT : 1)], B0[3 * (NAT > 0 ? NAT : 1)], A1[3 * (NAT > 0 ? NAT : 1)], B1[3 * (NAT > 0 ? NAT : 1)];
            load_evec<3 * NAT>(eA0, A0); load_evec<3 * NAT>(eB0, B0); load_evec<3 * NAT>(eA1, A1); load_evec<3 * NAT>(eB1, B1);
            contract_process2<NAT>(d, bs, A0, B0, premul(d, xc0), A1, B1, premul(d, xc1), V0, V1);
        } else {
            contract_process2_generic(d, bs, eA0, eB0, premul(d, xc0), eA1, eB1, premul(d, xc1), V0, V1);
        }
        if (act0) { sW += e0.w; sG = fma(e0.w, V0.x * V0.x + V0.y * V0.y, sG); }
        if (act1) { sW += e1.w; sG = fma(e1.w, V1.x * V1.x + V1.y * V1.y, sG); }
    }
    const double rowfac = rw.occ_row / rw.wrow;
    const double tG = block_sum<double>(sG, red);
    const double tW = block_sum<double>(sW, red);
    if (threadIdx.x == 0) {                                           // processes: both orderings of a listed pair count
        const uint4 pc = __ldg(reinterpret_cast<const uint4 *>(pcnt) + r);
        partial[r] = make_double2(rowfac * tG, rowfac * tW); counts[r] = pc.x + pc.y + pc.z + pc.w;
    }
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------------------------------
void launch_pre3(const FpDev &d, const IfcDev &f, const int32_t *targets, int64_t nt, double2 *mhat, cudaStream_t st) {
    if (nt > 0) k_pre3<<<(unsigned)nt, 256, 0, st>>>(d, f, targets, mhat);
}
void launch_pre4(const FpDev &d, const IfcDev &f, const int32_t *targets, int64_t nt, double2 *t0, cudaStream_t st) {
    if (nt > 0) k_pre4<<<(unsigned)nt, 256, 0, st>>>(d, f, targets, t0);
}

static size_t tables_smem_bytes(const FpDev &d, const IfcDev &f) {
    return (size_t)f.nblk * 9 * sizeof(double2) + (size_t)d.L * sizeof(double2) + (size_t)d.nb * sizeof(double2) +
           (size_t)f.nblk * sizeof(int4) + (size_t)((d.nat * d.nat + 1 + 3) & ~3) * sizeof(int);
}
size_t rates_smem_bytes(const FpDev &d, const IfcDev &f) {
    size_t b = tables_smem_bytes(d, f) + (size_t)(RW * QCAP + RW * 32) * sizeof(uint2) + (size_t)(RW * PCAP) * sizeof(uint32_t);
    return (b + 15) & ~(size_t)15;
}

// Dynamic shared memory above 48 KB needs an opt-in per kernel AND per device (the attribute is a per-device setting):
// the granted size is cached per (kernel instantiation, device), under a lock.
struct SmemGrant { std::mutex mu; size_t granted[64] = {}; };
template <typename K>
static cudaError_t opt_in_smem(K kernel, size_t smem, SmemGrant &g) {   // opt-in limit is 227 KB minus the static part
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

template <int ORDER, int NAT, int TILE>
static cudaError_t launch_rates_t(const FpDev &d, const IfcDev &f, const RowArgs &ra, int64_t nrows, const double2 *pre,
                                  double2 *partial, uint32_t *counts, bool only_flagged, cudaStream_t st) {
    const size_t smem = rates_smem_bytes(d, f);
    static SmemGrant granted;
    cudaError_t e = opt_in_smem(k_rates<ORDER, NAT, TILE>, smem, granted);
    if (e != cudaSuccess) return e;
    k_rates<ORDER, NAT, TILE><<<(unsigned)nrows, RT, smem, st>>>(d, f, ra, pre, partial, counts, only_flagged);
    return cudaGetLastError();
}

cudaError_t launch_rates(int order, const FpDev &d, const IfcDev &f, const RowArgs &ra, int64_t nrows, const double2 *pre,
                         double2 *partial, uint32_t *counts, bool only_flagged, cudaStream_t st) {
    if (nrows <= 0) return cudaSuccess;
    const bool t6 = d.nb % 6 == 0;
#define FP_ARGS d, f, ra, nrows, pre, partial, counts, only_flagged, st
    if (order == 3) {
        if (d.nat == 1) return launch_rates_t<3, 1, 3>(FP_ARGS);
        if (d.nat == 2) return launch_rates_t<3, 2, 6>(FP_ARGS);
        return t6 ? launch_rates_t<3, 0, 6>(FP_ARGS) : launch_rates_t<3, 0, 3>(FP_ARGS);
    }
    if (d.nat == 1) return launch_rates_t<4, 1, 3>(FP_ARGS);
    if (d.nat == 2) return launch_rates_t<4, 2, 6>(FP_ARGS);
    return t6 ? launch_rates_t<4, 0, 6>(FP_ARGS) : launch_rates_t<4, 0, 3>(FP_ARGS);
#undef FP_ARGS
}

// ---- split path ------------------------------------------------------------------------------------------------------
// entries one warp of k_enum can write for one row: its share of the sub-tile steps, every candidate admitted
int64_t enum_slot_entries(const FpDev &d) {
    const int tile = d.nb % 6 == 0 ? 6 : 3;
    const int64_t nsub = d.nb / tile, nsteps = (int64_t)((d.N + 31) >> 5) * nsub * nsub;
    return (nsteps + RW - 1) / RW * 32 * tile * tile;
}
int enum_warps_per_row() { return RW; }

cudaError_t launch_enum(int order, const FpDev &d, const RowArgs &ra, int64_t nrows, int64_t capw, ListEnt *lists,
                        uint32_t *wcnt, uint32_t *pcnt, cudaStream_t st) {
    if (nrows <= 0) return cudaSuccess;
    const unsigned g = (unsigned)nrows;
#define FP_ENUM(O, T, S) k_enum<O, T, S><<<g, RT, 0, st>>>(d, ra, capw, lists, wcnt, pcnt)
    if (order == 3) {
        if (d.nb == 6) FP_ENUM(3, 6, true); else if (d.nb == 3) FP_ENUM(3, 3, true);
        else if (d.nb % 6 == 0) FP_ENUM(3, 6, false); else FP_ENUM(3, 3, false);
    } else {
        if (d.nb == 6) FP_ENUM(4, 6, true); else if (d.nb == 3) FP_ENUM(4, 3, true);
        else if (d.nb % 6 == 0) FP_ENUM(4, 6, false); else FP_ENUM(4, 3, false);
    }
#undef FP_ENUM
    return cudaGetLastError();
}

template <int ORDER, int NAT>
static cudaError_t launch_eval_t(const FpDev &d, const IfcDev &f, const RowArgs &ra, int64_t nrows, const double2 *pre,
                                 int64_t capw, const ListEnt *lists, const uint32_t *wcnt, const uint32_t *pcnt,
                                 double2 *partial, uint32_t *counts, cudaStream_t st) {
    const size_t smem = (tables_smem_bytes(d, f) + 15) & ~(size_t)15;
    static SmemGrant granted;
    cudaError_t e = opt_in_smem(k_eval<ORDER, NAT>, smem, granted);
    if (e != cudaSuccess) return e;
    k_eval<ORDER, NAT><<<(unsigned)nrows, EVT, smem, st>>>(d, f, ra, pre, capw, lists, wcnt, pcnt, partial, counts);
    return cudaGetLastError();
}

cudaError_t launch_eval(int order, const FpDev &d, const IfcDev &f, const RowArgs &ra, int64_t nrows, const double2 *pre,
                        int64_t capw, const ListEnt *lists, const uint32_t *wcnt, const uint32_t *pcnt, double2 *partial,
                        uint32_t *counts, cudaStream_t st) {
    if (nrows <= 0) return cudaSuccess;
#define FP_ARGS d, f, ra, nrows, pre, capw, lists, wcnt, pcnt, partial, counts, st
    if (order == 3) {
        if (d.nat == 1) return launch_eval_t<3, 1>(FP_ARGS);
        if (d.nat == 2) return launch_eval_t<3, 2>(FP_ARGS);
        return launch_eval_t<3, 0>(FP_ARGS);
    }
    if (d.nat == 1) return launch_eval_t<4, 1>(FP_ARGS);
    if (d.nat == 2) return launch_eval_t<4, 2>(FP_ARGS);
    return launch_eval_t<4, 0>(FP_ARGS);
#undef FP_ARGS
}
