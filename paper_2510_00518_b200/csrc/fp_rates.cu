// fp_rates.cu -- the per-target pre-contraction and the fused rate kernel of the FourPhonon hot path (SURVEY.md §8(a)
// rows a2/a3 + a5/a6 + a7).
//
//   k_pre3/k_pre4  per-target level-0 contraction of the IFC list with the target eigenvector
//   group path (default): k_enum_g -> per-row process lists -> k_eval_g, in fp_group.cu
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
#include "fp_contract.cuh"

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
// a2/a3 + a5/a6 + a7: fused enumerate -> shared-memory queue -> evaluate
// ---------------------------------------------------------------------------------------------------------------------
constexpr int RATES_MINB = 4;                 // k_rates: 128 registers
constexpr int RT = 128;                       // threads per row CTA
constexpr int RW = RT / 32;                   // warps
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
                                                           RowWeights &rw, bool mglobal) {
    const bool mg = ORDER == 3 && mglobal;                            // Mhat stays in the level-0 table (global memory)
    bs.M = mg ? const_cast<double2 *>(pre) + (size_t)row.t * f.nblk * 9 : reinterpret_cast<double2 *>(smem_raw);
    bs.ph = reinterpret_cast<double2 *>(smem_raw) + (mg ? 0 : 9 * f.nblk);
    double2 *e1 = bs.ph + d.L;                                        // nb entries (level 1 of ORDER 4)
    bs.meta = reinterpret_cast<int4 *>(e1 + d.nb);
    bs.seg = reinterpret_cast<int *>(bs.meta + f.nblk);
    for (int i = threadIdx.x; i < f.nblk; i += blockDim.x) bs.meta[i] = f.blk_meta[i];
    for (int i = threadIdx.x; i <= d.nat * d.nat; i += blockDim.x) bs.seg[i] = f.seg[i];
    if (ORDER == 3) {
        const double2 *src = pre + (size_t)row.t * f.nblk * 9;
        if (!mg)
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
        float2 A = __ldg(pa + (size_t)i * d.N);                       // omega_f = NaN for zero modes: never admitted
        if (d.pfOff) A.y = __int_as_float(0x7f800000);               // fp_set_prefilter(ctx, 0): n' = inf
        const float ba = inq ? (row.s2 > 0 ? basef + A.x : basef - A.x) : fnan;
        lo[i] = ba - A.y; hi[i] = ba + A.y;
    }
    uint64_t mask = 0;
#pragma unroll
    for (int k = 0; k < TILE; k++) {
        float2 B = __ldg(pb + (size_t)k * d.N);
        if (d.pfOff) B.y = __int_as_float(0x7f800000);
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
    uint2 *evq = reinterpret_cast<uint2 *>(setup_row_tables<ORDER>(d, f, row, pre, smem_raw, bs, rw, ra.mglobal != 0));   // RW*QCAP
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

}  // namespace

// ---------------------------------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------------------------------
// ---------------------------------------------------------------------------------------------------------------------
// per-process terms (an iterative solver needs the rate of every single process)
// ---------------------------------------------------------------------------------------------------------------------
// One CTA per row of an explicit process list (k_count -> k_scan -> k_fill, fp_kernels.cu): the row's tables as in
// k_rates, then every listed process through the same eval_process -- pinned decision, weights, level-2 contraction --
// whose result is stored instead of summed: gamma_p = scale * WP_p |V_p|^2, scale = (C/N^k) x the channel's symmetry weight.
template <int ORDER>
__global__ void __launch_bounds__(RT) k_terms(FpDev d, IfcDev f, RowArgs ra, const double2 *pre, const int64_t *offsets,
                                              int64_t list_base, const uint32_t *list, double scale, double *gamma_p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int64_t r = ra.row0 + blockIdx.x;
    const int64_t beg = offsets[r] - list_base, cnt = offsets[r + 1] - offsets[r];
    if (cnt == 0) return;
    const Row row = make_row<ORDER>(d, ra, r);
    BlkSmem bs;
    RowWeights rw;
    setup_row_tables<ORDER>(d, f, row, pre, smem_raw, bs, rw, ra.mglobal != 0);
    for (int64_t i0 = 0; i0 < cnt; i0 += RT) {
        const int64_t i = i0 + threadIdx.x;
        const bool act = i < cnt;
        const uint32_t code = list[beg + (act ? i : 0)];
        const int p = (int)(code / (uint32_t)d.nb), jb = (int)(code - (uint32_t)p * (uint32_t)d.nb);
        const int qx = p / d.nb, ja = p - qx * d.nb;
        const int ql = q_index(d, q_add(d, row.qb, row.s2, unpack_qc(d.qc[qx])));
        double sG = 0.0, sW = 0.0;
        unsigned c = 0;
        eval_process<ORDER, 0>(d, bs, row, rw, make_uint2(((uint32_t)qx << 6) | (uint32_t)ja, ((uint32_t)ql << 6) | (uint32_t)jb), act, sG,
                               sW, c);
        if (act) gamma_p[beg + i] = scale * sG;
    }
}

void launch_pre3(const FpDev &d, const IfcDev &f, const int32_t *targets, int64_t nt, double2 *mhat, cudaStream_t st) {
    if (nt > 0) k_pre3<<<(unsigned)nt, 256, 0, st>>>(d, f, targets, mhat);
}
void launch_pre4(const FpDev &d, const IfcDev &f, const int32_t *targets, int64_t nt, double2 *t0, cudaStream_t st) {
    if (nt > 0) k_pre4<<<(unsigned)nt, 256, 0, st>>>(d, f, targets, t0);
}

static size_t tables_smem_bytes(const FpDev &d, const IfcDev &f, bool mglobal) {
    return (mglobal ? 0 : (size_t)f.nblk * 9 * sizeof(double2)) + (size_t)d.L * sizeof(double2) + (size_t)d.nb * sizeof(double2) +
           (size_t)f.nblk * sizeof(int4) + (size_t)((d.nat * d.nat + 1 + 3) & ~3) * sizeof(int);
}
cudaError_t launch_terms(int order, const FpDev &d, const IfcDev &f, const RowArgs &ra, int64_t nrows, const double2 *pre,
                         const int64_t *offsets, int64_t list_base, const uint32_t *list, double scale, double *gamma_p,
                         cudaStream_t st) {
    if (nrows <= 0) return cudaSuccess;
    const size_t smem = (tables_smem_bytes(d, f, ra.mglobal != 0) + 15) & ~(size_t)15;
    static SmemGrant g3, g4;
    if (order == 3) {
        cudaError_t e = opt_in_smem(k_terms<3>, smem, g3);
        if (e != cudaSuccess) return e;
        k_terms<3><<<(unsigned)nrows, RT, smem, st>>>(d, f, ra, pre, offsets, list_base, list, scale, gamma_p);
    } else {
        cudaError_t e = opt_in_smem(k_terms<4>, smem, g4);
        if (e != cudaSuccess) return e;
        k_terms<4><<<(unsigned)nrows, RT, smem, st>>>(d, f, ra, pre, offsets, list_base, list, scale, gamma_p);
    }
    return cudaGetLastError();
}
bool ifc_mglobal(const FpDev &d, const IfcDev &f, int order) { return order == 3 && rates_smem_bytes(d, f, false) > 226 * 1024; }
size_t rates_smem_bytes(const FpDev &d, const IfcDev &f, bool mglobal) {
    size_t b = tables_smem_bytes(d, f, mglobal) + (size_t)(RW * QCAP + RW * 32) * sizeof(uint2) + (size_t)(RW * PCAP) * sizeof(uint32_t);
    return (b + 15) & ~(size_t)15;
}

template <int ORDER, int NAT, int TILE>
static cudaError_t launch_rates_t(const FpDev &d, const IfcDev &f, const RowArgs &ra, int64_t nrows, const double2 *pre,
                                  double2 *partial, uint32_t *counts, bool only_flagged, cudaStream_t st) {
    const size_t smem = rates_smem_bytes(d, f, ra.mglobal != 0);
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
