// fp_group.cu -- the group path (the default of fp_rates3 / fp_rates4): Algorithm 3 -> Algorithm 4 of the paper
// (enumerate the allowed processes into index lists, then evaluate them), both halves on the device.
//
// Rows -- 3ph: (target, channel); 4ph: (target, channel, lambda') -- whose targets share their q-point (and, for 4ph,
// whose lambda' share q') have the same q_base, hence the same momentum map q_A -> q_B and the same
// records of the two free legs A, B; they differ only in their base energy Obase = omega (3ph) or omega +- omega' (4ph).
//
//   k_enum_g   one CTA per group of up to FP_GROUP_RMAX such rows.  The base energies are sorted once.  Every lane owns
//              one q_A of a 32-point tile and tests each (j_A, j_B) pair ONCE for all rows: an FP32 bound of the window
//              half-width (bnd >= ncut sigma + rounding slack) gives the interval of base energies that
//              can pass, a bisection over the sorted base energies gives the rows inside it.  The (row, pair) survivors
//              are queued in shared memory and, 32 at a time, take the window decision in the pinned
//              FP64 arithmetic of SURVEY.md §8(c) step 3 -- which alone determines counts and rates -- and the
//              row-independent part of the weight; allowed processes go to the list slot of their
//              row (16 bytes per process), in a deterministic order.
//   k_eval_g   one CTA per tile of rows of a group: level 1 of the contraction for all rows of the tile (the rows of
//              one target share the loads of its level-0 table), then the matrix element of every listed process
//              (compute_Vp), two processes per lane against one pass over the row's contraction
//              blocks, in 64-process chunks dealt round-robin to the warps; fixed-order row sums.
#include <algorithm>

#include "fp_contract.cuh"

namespace {

constexpr int GW = 4;                         // warps per CTA (both kernels)
#ifndef FP_ENUM_NU
#define FP_ENUM_NU 16
#endif
constexpr int NUMAX = FP_ENUM_NU;             // enumeration units (shares of the q_A tiles) = list slots per row: ga.nu, a
                                              // power of two <= NUMAX (and <= the number of tiles)
constexpr int GT = GW * 32;
constexpr int RMAX = FP_GROUP_RMAX;           // rows per enumerator group
#ifndef FP_ENUM_QC
#define FP_ENUM_QC 2048         // measured (B200): 1024 / 1536 / 2048 / 2560 -> k_enum_g 249 / 244 / 243 / 298 ms at config 3 (2560 costs a CTA per SM), 504 / 479 / 457 / 452 ms at config 4
#endif
#ifndef FP_ENUM_MINB
#define FP_ENUM_MINB 6
#endif
constexpr int QC = FP_ENUM_QC;                // survivor queue of a warp; drained when the next j_A iteration may not fit
static_assert(RMAX == 64, "the bisection of k_enum_g is written for 64 sorted base energies");
static_assert(6 * RMAX <= QC, "one lane's survivors of one j_A iteration (TB <= 6 branches x RMAX rows) must fit the queue");
constexpr unsigned SLOT_FULL = 0xffffffffu;   // entry count of a list slot that filled up

struct Group {
    int g, ch, qi, s1, s2, q1;                // group, channel, q' index (4ph), signs, q' (4ph)
    int m0, R, j0, nj;                        // first member (offset into gmem), rows of the group, j' range (4ph)
    int3 qb;                                  // base q coordinates: q (3ph) or q + s1 q' (4ph)
};

template <int ORDER>
__device__ __forceinline__ Group decode_group(const FpDev &d, const GroupArgs &ga, int64_t gid) {
    Group G;
    if (ORDER == 3) {
        G.g = (int)(gid >> 1); G.ch = (int)(gid & 1); G.qi = 0; G.q1 = -1;
        G.s1 = +1; G.s2 = G.ch == 0 ? +1 : -1;
    } else {
        G.qi = (int)(gid % ga.nqp); gid /= ga.nqp;
        G.ch = (int)(gid % 3); G.g = (int)(gid / 3);
        G.q1 = ga.qp_begin + G.qi;
        G.s1 = G.ch == 2 ? -1 : +1; G.s2 = G.ch == 0 ? +1 : -1;
    }
    const int4 gd = ga.gdesc[G.g];
    G.m0 = gd.y; G.j0 = gd.w & 0xffff; G.nj = gd.w >> 16;
    G.R = ORDER == 3 ? gd.z : gd.z * G.nj;
    const int3 qg = unpack_qc(d.qc[gd.x]);
    G.qb = ORDER == 3 ? qg : q_add(d, qg, G.s1, unpack_qc(d.qc[G.q1]));
    return G;
}

// row rr of a group -> local target index, lambda' (4ph), index of the row in the per-row arrays (the order of
// make_row / k_rates / k_finalize: 3ph t*2 + ch; 4ph ((t*3 + ch)*nqp + qi)*nb + j')
template <int ORDER>
__device__ __forceinline__ void group_row(const FpDev &d, const GroupArgs &ga, const Group &G, int rr, int &t, int &lam1,
                                          int64_t &rold) {
    if (ORDER == 3) {
        t = ga.gmem[G.m0 + rr]; lam1 = -1;
        rold = (int64_t)t * 2 + G.ch;
    } else {
        const int m = rr / G.nj, j1 = G.j0 + rr - m * G.nj;
        t = ga.gmem[G.m0 + m]; lam1 = G.q1 * d.nb + j1;
        rold = (((int64_t)t * 3 + G.ch) * ga.nqp + G.qi) * d.nb + j1;
    }
}

// exp(x) for the Gaussian weight: allowed processes have x = -(Delta/sigma)^2 in [-ncut^2, 0], so for
// x in [-8, 0] a short kernel serves -- n = rint(x log2 e), f = x - n ln 2 (two-term), degree-11 Taylor polynomial of
// exp(f) on |f| <= 0.347 (truncation 6e-15 relative), scaled by 2^n through the exponent field; anything else takes exp().
__device__ __forceinline__ double exp_window(double x) {
    if (!(x >= -8.0)) return exp(x);
    const double t = fma(x, 1.4426950408889634074, 6755399441055744.0);
    const int n = __double2loint(t);
    const double dn = t - 6755399441055744.0;
    double f = fma(dn, -6.93147180369123816490e-01, x);
    f = fma(dn, -1.90821492927058770002e-10, f);
    double p = 2.5052108385441718775e-08;                              // 1/11!
    p = fma(p, f, 2.7557319223985890653e-07);
    p = fma(p, f, 2.7557319223985892511e-06);
    p = fma(p, f, 2.4801587301587301566e-05);
    p = fma(p, f, 1.9841269841269841253e-04);
    p = fma(p, f, 1.3888888888888889419e-03);
    p = fma(p, f, 8.3333333333333332177e-03);
    p = fma(p, f, 4.1666666666666664354e-02);
    p = fma(p, f, 1.6666666666666665741e-01);
    p = fma(p, f, 0.5);
    p = fma(p, f, 1.0);
    p = fma(p, f, 1.0);
    return __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));
}

// ---------------------------------------------------------------------------------------------------------------------
// a2 / a3 + a7: group enumerator
// ---------------------------------------------------------------------------------------------------------------------
// Persistent and warp-autonomous: the work of a launch is cut into units (group CTA gl, share u of its q_A tiles:
// tiles u, u + NU, ...), dealt to the warps through an atomic counter.  Unit (gl, u) owns list slot u of every row of
// gl, so what is written where does not depend on which warp ran the unit: lists are reproducible run to run.
// queue entry: lane that owns q_A (5 bits) | j_A << 5 (6 bits) | j_B << 11 (6 bits) | sorted row index << 17 (7 bits)
struct EnumWarpSmem {
    double Sd[RMAX];                          // base energies of the group's rows, sorted ascending (the pinned values)
    float Sf[RMAX + 4];                       // ... rounded to FP32, padded with +inf
    unsigned char Srr[RMAX];                  // sorted index -> row rr
    unsigned cnt[RMAX];                       // entries written per row (this unit's slot)
    int ql[32];                               // q_B of the tile's 32 q_A
    uint32_t pend[QC];                        // survivor queue
};

template <int ORDER, int TB>
__global__ void __launch_bounds__(GT, FP_ENUM_MINB) k_enum_g(FpDev d, GroupArgs ga, int64_t ngc, int64_t capw, ListEnt *lists,
                                                            uint32_t *wcnt, unsigned int *work) {
    __shared__ EnumWarpSmem sm_all[GW];
    EnumWarpSmem &sm = sm_all[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const int nb = d.nb;
    const int ntiles = (d.N + 31) >> 5;
    const float fnan = __int_as_float(0x7fc00000), finf = __int_as_float(0x7f800000);
    const int NU = ga.nu;
    const int64_t nunits = ngc * NU;
    unsigned nadm = 0, nent = 0;                                      // statistics (profiling)

    for (;;) {
        int64_t unit = 0;
        if (lane == 0) unit = (int64_t)atomicAdd(work, 1u);
        unit = __shfl_sync(0xffffffffu, unit, 0);
        if (unit >= nunits) break;
        const int64_t gl = unit / NU;
        const int u = (int)(unit - gl * NU);
        const Group G = decode_group<ORDER>(d, ga, ga.gid0 + gl);

        // ---- rows of the group, sorted by base energy (two rows per lane) ------------------------------------------------
        double ob[2];
#pragma unroll
        for (int h = 0; h < 2; h++) {
            const int rr = lane + 32 * h;
            ob[h] = __longlong_as_double(0x7ff8000000000000ll);      // NaN: not a row, or a zero mode is a leg (item 8)
            if (rr < G.R) {
                int t, lam1; int64_t rold;
                group_row<ORDER>(d, ga, G, rr, t, lam1, rold);
                const double w = d.rec[ga.targets[t]].omega;
                if (ORDER == 3) { if (w != 0.0) ob[h] = w; }
                else {
                    const double w1 = d.rec[lam1].omega;                  // pinned: Obase = fl(omega +- omega')
                    if (w != 0.0 && w1 != 0.0) ob[h] = G.s1 > 0 ? __dadd_rn(w, w1) : __dsub_rn(w, w1);
                }
            }
            sm.cnt[rr] = 0;
            sm.Sf[rr] = finf;
        }
        if (lane < 4) sm.Sf[RMAX + lane] = finf;
        const int nvalid = __popc(__ballot_sync(0xffffffffu, ob[0] == ob[0])) + __popc(__ballot_sync(0xffffffffu, ob[1] == ob[1]));
        __syncwarp();
        {
            int rank[2] = {0, 0};
            for (int k = 0; k < 64; k++) {
                const double o = __shfl_sync(0xffffffffu, ob[k >> 5], k & 31);
#pragma unroll
                for (int h = 0; h < 2; h++) rank[h] += (o < ob[h] || (o == ob[h] && k < lane + 32 * h)) ? 1 : 0;
            }
#pragma unroll
            for (int h = 0; h < 2; h++)
                if (ob[h] == ob[h]) { sm.Sd[rank[h]] = ob[h]; sm.Sf[rank[h]] = (float)ob[h]; sm.Srr[rank[h]] = (unsigned char)(lane + 32 * h); }
        }
        __syncwarp();

        if (nvalid > 0) {
            const float Smin = sm.Sf[0], Smax = sm.Sf[nvalid - 1];
            int top = 1;                                              // first bisection step: largest power of two < nvalid + 1
            while (2 * top <= nvalid) top *= 2;
            const bool sym = ga.sym && G.s2 < 0;                      // pair symmetry: list mode A <= mode B only
            int wp = 0;

            ListEnt *ubase = lists + ((size_t)gl * ga.rmaxg * NU + u) * (size_t)capw;   // slot u of row 0 of this group CTA
            const unsigned rowstride = (unsigned)NU * (unsigned)capw;
            // stage 3 of every queued survivor of the current tile: the pinned decision and the weight
            auto drain = [&](int tile, int n) {
                for (int base = 0; base < n; base += 32) {
                    const bool in = base + lane < n;
                    const uint32_t e = sm.pend[base + (in ? lane : 0)];
                    const int src = (int)(e & 31u), ja = (int)((e >> 5) & 63u), jb = (int)((e >> 11) & 63u), k = (int)(e >> 17);
                    const int qx = (tile << 5) + src, ql = sm.ql[src];
                    const int p = qx * nb + ja, lamB = ql * nb + jb;
                    const ModeRec a = load_rec(d.rec + p), b = load_rec(d.rec + lamB);
                    const double2 xa = __ldg(d.aux + p), xb = __ldg(d.aux + lamB);
                    const double O = sm.Sd[k];
                    const int rr = sm.Srr[k];
                    // sigma (compute_sigma): the sum of squares in the pinned order; the square root and the
                    // division only where the fast comparison cannot decide (relative margin 1e-13, error of the fast
                    // threshold < 2e-15)
                    double s, thr, inv;
                    if (d.sigma_const > 0.0) { s = 1.0; thr = __dmul_rn(d.ncut, d.sigma_const); inv = d.invC; }
                    else {
                        const double dx = __dsub_rn(a.vx, b.vx), dy = __dsub_rn(a.vy, b.vy), dz = __dsub_rn(a.vz, b.vz);
                        const double t0 = __dadd_rn(__dadd_rn(__dmul_rn(d.B[0], dx), __dmul_rn(d.B[1], dy)), __dmul_rn(d.B[2], dz));
                        const double t1 = __dadd_rn(__dadd_rn(__dmul_rn(d.B[3], dx), __dmul_rn(d.B[4], dy)), __dmul_rn(d.B[5], dz));
                        const double t2 = __dadd_rn(__dadd_rn(__dmul_rn(d.B[6], dx), __dmul_rn(d.B[7], dy)), __dmul_rn(d.B[8], dz));
                        s = __dadd_rn(__dadd_rn(__dmul_rn(t0, t0), __dmul_rn(t1, t1)), __dmul_rn(t2, t2));
                        const double r = rsqrt(s);
                        thr = d.thrC * (s * r);
                        inv = r * d.invC;
                    }
                    const double thr_lo = thr * (1.0 - 1e-13), thr_hi = thr * (1.0 + 1e-13);
                    auto decide = [&](double delta) -> bool {         // == (sigma > 0 && |delta| <= ncut * sigma), pinned
                        const double ad = fabs(delta);
                        if (!(s > 0.0)) return false;
                        if (ad <= thr_lo) return true;
                        if (ad > thr_hi) return false;
                        const double sig = d.sigma_const > 0.0 ? d.sigma_const : __dmul_rn(d.scale, __dsqrt_rn(__ddiv_rn(s, 6.0)));
                        return sig > 0.0 && ad <= __dmul_rn(d.ncut, sig);
                    };
                    const bool legs = in && a.omega != 0.0 && b.omega != 0.0;
                    const double delta = __dsub_rn(G.s2 > 0 ? __dadd_rn(O, a.omega) : __dsub_rn(O, a.omega), b.omega);
                    bool ok = legs && decide(delta);
                    // weight without the row factors: occ(f_A, f_B) g / (omega_A omega_B), g = exp(-(Delta/sigma)^2)/(sigma sqrt(pi))
                    double occ;
                    if (ORDER == 3) occ = G.s2 > 0 ? (xa.x - xb.x) : (xa.x + xb.x + 1.0);   // symmetric in (A, B) for s2 < 0
                    else occ = (G.s2 > 0 ? 1.0 + xa.x : xa.x) * xb.x;
                    const double pf = occ * (xa.y * xb.y) * (inv * 0.56418958354775628695);   // 1/sqrt(pi)
                    const double r1 = delta * inv;
                    const double g1 = exp_window(-(r1 * r1));
                    double w = ok ? pf * g1 : 0.0;
                    bool two = false;
                    if (sym) {                                        // the other ordering: Delta' = (Obase - omega_B) - omega_A
                        const double delta2 = __dsub_rn(__dsub_rn(O, b.omega), a.omega);
                        const bool ok2 = legs && p != lamB && decide(delta2);   // (A = B is its own partner: one process)
                        if (ok2) {
                            const double dd = (delta2 - delta) * inv; // the two Delta differ by rounding only
                            const double g2 = fabs(dd) < 1e-7 ? g1 * (1.0 - dd * (r1 + r1 + dd)) : exp_window(-((r1 + dd) * (r1 + dd)));
                            w += pf * g2;
                        }
                        two = ok && ok2;
                        ok = ok || ok2;
                    }
                    // ordered append to the slot of (row, unit): rank among the lanes of the batch with the same row
                    const unsigned peers = __match_any_sync(0xffffffffu, ok ? rr : RMAX + lane);
                    const unsigned rank = __popc(peers & ((1u << lane) - 1u));
                    unsigned basec = 0;
                    if (ok) basec = sm.cnt[rr];
                    __syncwarp();
                    if (ok) {
                        const unsigned npeer = __popc(peers);
                        if (basec == SLOT_FULL || basec + npeer > (unsigned)capw) {   // the slot of this row is full: the
                            if (rank == 0) sm.cnt[rr] = SLOT_FULL;                    // row (alone) is redone by k_rates
                        } else {
                            ListEnt en;
                            en.x = ((uint32_t)qx << 6) | (uint32_t)ja | (two ? 0x80000000u : 0u);
                            en.y = ((uint32_t)ql << 6) | (uint32_t)jb;
                            en.w = w;
                            ubase[(size_t)((unsigned)rr * rowstride) + basec + rank] = en;
                            if (rank == 0) sm.cnt[rr] = basec + npeer;
                            nent++;
                        }
                    }
                    __syncwarp();
                }
            };

            int tile = u, jb0s = 0, jas = 0, lane0s = 0;              // (jb0s, jas, lane0s): where to resume a tile after a drain
            while (tile < ntiles) {
                const int qx = (tile << 5) + lane;
                const bool inq = qx < d.N;
                const int qs = inq ? qx : 0;
                const int ql = q_index(d, q_add(d, G.qb, G.s2, unpack_qc(d.qc[qs])));
                {   // tile vote before any record is loaded: the frequency ranges of q_A and q_B (table qmm) bound
                    // c = omega_B - s2 omega_A, and a pair can pass only if [c - bnd, c + bnd] meets [Smin, Smax]
                    const float2 mA = __ldg(d.qmm + qs), mB = __ldg(d.qmm + ql);
                    const float clo = G.s2 > 0 ? mB.x - mA.y : mA.x + mB.x, chi = G.s2 > 0 ? mB.y - mA.x : mA.y + mB.y;
                    const bool live = inq && chi + d.gfW >= Smin && clo - d.gfW <= Smax && (!sym || qs <= ql);
                    if (!__any_sync(0xffffffffu, live)) { tile += NU; continue; }
                }
                sm.ql[lane] = ql;
                __syncwarp();
                const float4 *pa = d.recf + (size_t)qs * nb, *pb = d.recf + (size_t)ql * nb;
                const bool lane_ok = inq && (!sym || qs <= ql);
                bool redo = false;
                for (int jb0 = jb0s; jb0 < nb && !redo; jb0 += TB) {
                    float4 Bf[TB];
#pragma unroll
                    for (int k = 0; k < TB; k++) Bf[k] = __ldg(pb + jb0 + k);
                    const int ja_first = jb0 == jb0s ? jas : 0;
                    float4 An = __ldg(pa + ja_first);
                    for (int ja = ja_first; ja < nb; ja++) {
                        const float4 A = An;                          // omega_f = NaN for zero modes: never admitted
                        if (ja + 1 < nb) An = __ldg(pa + ja + 1);
                        const bool done = lane < lane0s && ja == jas && jb0 == jb0s;   // (queued by an earlier slice)
                        const float xa = lane_ok && !done ? (G.s2 > 0 ? A.x : -A.x) : fnan;
                        int kc[TB];
                        int ctot = 0;
#pragma unroll
                        for (int k = 0; k < TB; k++) {
                            const float4 B = Bf[k];
                            const float dx = A.y - B.y, dy = A.z - B.z, dz = A.w - B.w;
                            float rt;
                            asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(rt) : "f"(fmaf(dz, dz, fmaf(dy, dy, dx * dx))));
                            const float bnd = fminf(fmaf(d.gfC, rt, d.gfD), 1.0e38f);   // (finite: +inf is the padding of Sf)
                            float c = B.x - xa;                       // Obase + s2 omega_A - omega_B = 0  <=>  Obase = c
                            if (sym && qs == ql && ja > jb0 + k) c = fnan;
                            const float lo = c - bnd, hi = c + bnd;
                            int k0 = 0;                               // first sorted row with Sf >= lo
#pragma unroll
                            for (int st = RMAX / 2; st > 0; st >>= 1)
                                if (st <= top) k0 += (sm.Sf[k0 + st - 1] < lo) ? st : 0;
                            k0 += (sm.Sf[k0] < lo) ? 1 : 0;
                            int cn = 0;                               // (+inf padding ends the scan; NaN never starts it)
                            while (sm.Sf[k0 + cn] <= hi) cn++;
                            kc[k] = k0 | (cn << 8);
                            ctot += cn;
                        }
                        unsigned incl = (unsigned)ctot;               // ordered append to the survivor queue
#pragma unroll
                        for (int o = 1; o < 32; o <<= 1) {
                            const unsigned v = __shfl_up_sync(0xffffffffu, incl, o);
                            if (lane >= o) incl += v;
                        }
                        const int tot = (int)__shfl_sync(0xffffffffu, incl, 31);
                        if (tot == 0) continue;
                        if (wp + tot > QC) {                          // (only with very wide windows) drain, then resume
                            if (wp > 0) { redo = true; jb0s = jb0; jas = ja; lane0s = 0; break; }   // ... with this iteration
                            // One iteration alone exceeds the queue: it goes through in slices of whole lanes (a lane
                            // queues at most TB * RMAX <= QC survivors; the lanes below lane0s went in earlier slices),
                            // which keeps the order of every row's entries -- (j_B tile, j_A, lane, j_B, row) -- exactly
                            // what one big queue would give.
                            const int l1 = __popc(__ballot_sync(0xffffffffu, incl <= (unsigned)QC));   // incl is monotone
                            if (lane < l1) {
                                nadm += (unsigned)ctot;
                                int pos = (int)incl - ctot;
#pragma unroll
                                for (int k = 0; k < TB; k++) {
                                    const int k0 = kc[k] & 255, cn = kc[k] >> 8;
                                    for (int i = 0; i < cn; i++)
                                        sm.pend[pos++] = (uint32_t)lane | ((uint32_t)ja << 5) | ((uint32_t)(jb0 + k) << 11) | ((uint32_t)(k0 + i) << 17);
                                }
                            }
                            wp = (int)__shfl_sync(0xffffffffu, incl, l1 - 1);
                            redo = true; jb0s = jb0; jas = ja; lane0s = l1;
                            break;
                        }
                        nadm += (unsigned)ctot;
                        int pos = wp + (int)incl - ctot;
#pragma unroll
                        for (int k = 0; k < TB; k++) {
                            const int k0 = kc[k] & 255, cn = kc[k] >> 8;
                            for (int i = 0; i < cn; i++)
                                sm.pend[pos++] = (uint32_t)lane | ((uint32_t)ja << 5) | ((uint32_t)(jb0 + k) << 11) | ((uint32_t)(k0 + i) << 17);
                        }
                        wp += tot;
                    }
                }
                __syncwarp();
                drain(tile, wp);
                wp = 0;
                if (!redo) { tile += NU; jb0s = 0; jas = 0; lane0s = 0; }
            }
        }
        // ---- entry counts of this unit's slots (SLOT_FULL marks a row for the redo pass) -------------------------------
        __syncwarp();
        unsigned nfull = 0;
        for (int rr = lane; rr < ga.rmaxg; rr += 32) {
            const unsigned c = sm.cnt[rr];
            wcnt[((size_t)gl * ga.rmaxg + rr) * NU + u] = c;
            nfull += c == SLOT_FULL ? 1u : 0u;
        }
        if (__any_sync(0xffffffffu, nfull != 0) && nfull) atomicAdd(ga.overflow, nfull);
        __syncwarp();
    }
    if (ga.evaluated) {                                               // profiling only
        for (int o = 16; o > 0; o >>= 1) { nent += __shfl_down_sync(0xffffffffu, nent, o); nadm += __shfl_down_sync(0xffffffffu, nadm, o); }
        if (lane == 0) {
            if (nent) atomicAdd(ga.evaluated, (unsigned long long)nent);
            if (nadm) atomicAdd(ga.prefiltered, (unsigned long long)nadm);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// a5 / a6 + a8: tile evaluator
// ---------------------------------------------------------------------------------------------------------------------
struct EvalSmem {
    double2 *M;        // ge * nblk*9    Mhat of every row of the tile
    double2 *ph;       // L
    double2 *e1;       // ge * nb        level-1 eigenvectors (4ph)
    int4 *meta;        // nblk
    int *seg;          // nat*nat+1 (padded to 4)
    unsigned *rpre;    // ge * (NU + 1)  prefix sums of the NU slot lengths of a row: its slots read as one list
    double *rowfac;    // ge             row factors of the weight: occ_row / (omega [omega'])
    long long *rold;   // ge             index of the row in partial[] / counts[]
    int *chunk0;       // ge + 1         first 64-process chunk of each row
    double *accG, *accW;   // nw * ge    per (warp, row) sums
    unsigned *accC;    // nw * ge        processes (both orderings of a listed pair count)
    unsigned char *rot;  // ge           rotation of the row's chunk deal (a property of the row alone)
    double2 *As;       // nw * nb * 64   generic atom count: leg-A eigenvectors of a warp's chunk, [component][process]
    float2 *Mf, *phf;  // ge * nblk*9, L mixed precision: Mhat and the phases rounded to FP32
};
// nw = warps of the CTA; stage: the generic evaluator (NAT = 0) stages one eigenvector per process of every warp's chunk
// mg: the Mhat tables stay in global memory (3ph, IFC3 lists too long for shared memory)
__host__ __device__ inline size_t eval_smem_layout(int ge, int nblk, int L, int nb, int nat, int NU, int nw, bool stage, bool mixed,
                                                   EvalSmem *es, unsigned char *base, bool mg = false) {
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t r = o; o += (bytes + 15) & ~(size_t)15; return r; };
    const size_t oM = take(mg ? 0 : (size_t)ge * nblk * 9 * sizeof(double2)), oph = take((size_t)L * sizeof(double2)),
                 oe1 = take((size_t)ge * nb * sizeof(double2)), ometa = take((size_t)nblk * sizeof(int4)),
                 oseg = take((size_t)(nat * nat + 1) * sizeof(int)), orowp = take((size_t)ge * (NU + 1) * sizeof(unsigned)),
                 orf = take((size_t)ge * sizeof(double)), oro = take((size_t)ge * sizeof(long long)),
                 och = take((size_t)(ge + 1) * sizeof(int)), oaG = take((size_t)nw * ge * sizeof(double)),
                 oaW = take((size_t)nw * ge * sizeof(double)), oaC = take((size_t)nw * ge * sizeof(unsigned)),
                 orot = take((size_t)ge), oAs = take(stage ? (size_t)nw * nb * 64 * sizeof(double2) : 0),
                 oMf = take(mixed ? (size_t)ge * nblk * 9 * sizeof(float2) : 0), ophf = take(mixed ? (size_t)L * sizeof(float2) : 0);
    if (es) {
        es->M = reinterpret_cast<double2 *>(base + oM); es->ph = reinterpret_cast<double2 *>(base + oph);
        es->e1 = reinterpret_cast<double2 *>(base + oe1); es->meta = reinterpret_cast<int4 *>(base + ometa);
        es->seg = reinterpret_cast<int *>(base + oseg); es->rpre = reinterpret_cast<unsigned *>(base + orowp);
        es->rowfac = reinterpret_cast<double *>(base + orf); es->rold = reinterpret_cast<long long *>(base + oro);
        es->chunk0 = reinterpret_cast<int *>(base + och); es->accG = reinterpret_cast<double *>(base + oaG);
        es->accW = reinterpret_cast<double *>(base + oaW); es->accC = reinterpret_cast<unsigned *>(base + oaC);
        es->rot = base + orot; es->As = reinterpret_cast<double2 *>(base + oAs);
        es->Mf = reinterpret_cast<float2 *>(base + oMf); es->phf = reinterpret_cast<float2 *>(base + ophf);
    }
    return o;
}

#ifndef FP_EVAL_MINB
#define FP_EVAL_MINB 3
#endif
constexpr int GEN_WMAX = 8;                   // warps of a generic-evaluator CTA, at most (as many as the staging leaves room for)
// MIX: level-2 contraction in FP32 (fp_set_precision; NAT > 0 only)
// MG:  3ph only: Mhat of a row is read from the level-0 table in global memory, not from a shared-memory copy
template <int ORDER, int NAT, bool MIX, bool MG = false>
__global__ void __launch_bounds__(NAT > 0 ? GT : GEN_WMAX * 32, NAT > 0 ? (MIX ? 4 : FP_EVAL_MINB) : 1) k_eval_g(FpDev d, IfcDev f, GroupArgs ga, const double2 *pre, int64_t capw,
                                                  const ListEnt *lists, const uint32_t *wcnt, int ge, int tiles_per_group,
                                                  double2 *partial, uint32_t *counts) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int s_nitems;
    EvalSmem es;
    const int nthr = NAT > 0 ? GT : (int)blockDim.x, nw = nthr >> 5;  // (the generic evaluator picks its CTA size at launch)
    static_assert(!MG || (ORDER == 3 && !MIX), "global-memory Mhat: 3ph, FP64 only");
    eval_smem_layout(ge, f.nblk, d.L, d.nb, d.nat, ga.nu, nw, NAT == 0, MIX, &es, smem_raw, MG);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nb = d.nb;
    const int NU = ga.nu;
    const int64_t gl = blockIdx.x / tiles_per_group;
    const int rr0 = (int)(blockIdx.x - gl * tiles_per_group) * ge;
    const Group G = decode_group<ORDER>(d, ga, ga.gid0 + gl);
    const int nrt = min(ge, G.R - rr0);                               // rows of this tile
    if (nrt <= 0) return;

    // ---- the rows of the tile: list lengths, row factors ----------------------------------------------------------------
    for (int rt = threadIdx.x; rt < nrt; rt += nthr) {
        int t, lam1; int64_t rold;
        group_row<ORDER>(d, ga, G, rr0 + rt, t, lam1, rold);
        bool ovf = false;
        unsigned total = 0;
        es.rpre[rt * (NU + 1)] = 0;
        for (int k = 0; k < NU; k++) {
            const unsigned c = __ldg(wcnt + ((size_t)gl * ga.rmaxg + rr0 + rt) * NU + k);
            ovf = ovf || c == 0xffffffffu;
            total += c;
            es.rpre[rt * (NU + 1) + k + 1] = total;
        }
        if (ovf) { total = 0; es.rpre[rt * (NU + 1) + NU] = 0; }
        es.rold[rt] = rold;
        es.rot[rt] = (unsigned char)((unsigned)(ORDER == 3 ? ga.targets[t] : ga.targets[t] + lam1) % (unsigned)nw);
        const int lam = ga.targets[t];
        double fac = 0.0;
        if (total > 0) {
            const double w = d.rec[lam].omega;
            if (ORDER == 3) fac = 1.0 / w;
            else {
                const double f1 = d.occ[lam1];
                fac = ((G.s1 > 0 ? 1.0 + f1 : f1) / d.occ[lam]) / (w * d.rec[lam1].omega);
            }
        }
        es.rowfac[rt] = fac;
        if (total == 0) {                                             // (0xffffffff marks the row for the redo pass)
            partial[rold] = make_double2(0.0, 0.0);
            counts[rold] = ovf ? 0xffffffffu : 0u;
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int run = 0;
        for (int rt = 0; rt < nrt; rt++) { es.chunk0[rt] = run; run += (int)((es.rpre[rt * (NU + 1) + NU] + 63u) >> 6); }
        es.chunk0[nrt] = run;
        s_nitems = run;
    }
    __syncthreads();
    const int nitems = s_nitems;
    if (nitems == 0) return;

    // ---- tables of the tile: block metadata, level 1 for every row with a list ---------------------------------------------
    const int nm9 = f.nblk * 9;
    for (int i = threadIdx.x; i < f.nblk; i += nthr) {
        const int4 m = f.blk_meta[i];
        es.meta[i] = m;
    }
    for (int i = threadIdx.x; i <= d.nat * d.nat; i += nthr) es.seg[i] = f.seg[i];
    if (ORDER == 3) {
        for (int rt = 0; rt < nrt; rt++) {
            if (es.rpre[rt * (NU + 1) + NU] == 0) continue;
            int t, lam1; int64_t rold;
            group_row<ORDER>(d, ga, G, rr0 + rt, t, lam1, rold);
            const double2 *src = pre + (size_t)t * nm9;
            if (!MG)
                for (int i = threadIdx.x; i < nm9; i += nthr) es.M[rt * nm9 + i] = src[i];
        }
    } else {
        // level 1: Mhat_b[x][y] = sum_{c in b} phi(s1 q', Rj-Rl) sum_be T0[c][be][x][y] A'(j_c, be), A' = e~ (s1=+) or conj
        for (int i = threadIdx.x; i < d.L; i += nthr) {
            double2 p = d.ph1d[i];
            if (G.s1 < 0) p.y = -p.y;
            es.ph[i] = p;
        }
        for (int i = threadIdx.x; i < nrt * nb; i += nthr) {
            const int rt = i / nb, c = i - rt * nb;
            const int j1 = G.j0 + (rr0 + rt) % G.nj;
            es.e1[i] = (G.s1 > 0 ? d.evec : d.evecc)[((size_t)G.q1 * nb + j1) * nb + c];
        }
        __syncthreads();
        const int3 qm1 = premul(d, unpack_qc(d.qc[G.q1]));
        // rows of one target share the loads of its T0: work item = (member of the tile, output element), inner loop
        // over that member's rows (at most nb)
        const int nj = G.nj;
        const int m_lo = rr0 / nj, m_hi = (rr0 + nrt - 1) / nj;
        for (int o = threadIdx.x; o < (m_hi - m_lo + 1) * nm9; o += nthr) {
            const int mi = o / nm9, bo = o - mi * nm9;
            const int b = bo / 9, xy = bo - 9 * b;
            const int m = m_lo + mi;
            const int rt_lo = max(m * nj, rr0) - rr0, rt_hi = min((m + 1) * nj, rr0 + nrt) - rr0;   // rows [rt_lo, rt_hi)
            const int t = ga.gmem[G.m0 + m];
            const double2 *T0 = pre + (size_t)t * f.n * 27;
            for (int r0 = rt_lo; r0 < rt_hi; r0 += 6) {
                const int nr = min(6, rt_hi - r0);
                double2 acc[6];
#pragma unroll
                for (int k = 0; k < 6; k++) acc[k] = make_double2(0.0, 0.0);
                for (int c = f.blk_start[b]; c < f.blk_start[b + 1]; c++) {
                    const int4 m1 = f.cl_meta1[c];
                    const double2 ph = es.ph[phase_idx(d, qm1, m1.y, m1.z, m1.w)];
                    double2 tv[3];
#pragma unroll
                    for (int be = 0; be < 3; be++) tv[be] = cmul(T0[(size_t)c * 27 + 9 * be + xy], ph);
#pragma unroll
                    for (int k = 0; k < 6; k++)
                        if (k < nr) {
                            const double2 *e = es.e1 + (r0 + k) * nb + 3 * m1.x;
#pragma unroll
                            for (int be = 0; be < 3; be++) cfma(acc[k], tv[be], e[be]);
                        }
                }
#pragma unroll
                for (int k = 0; k < 6; k++)
                    if (k < nr) es.M[(r0 + k) * nm9 + bo] = acc[k];
            }
        }
        __syncthreads();
    }
    for (int i = threadIdx.x; i < d.L; i += nthr) {                     // phases of the free legs: phi(s2 qx, dR)
        double2 p = d.ph1d[i];
        if (G.s2 < 0) p.y = -p.y;
        es.ph[i] = p;
        if (MIX) es.phf[i] = make_float2((float)p.x, (float)p.y);
    }
    __syncthreads();
    if (MIX) {                                                        // (after the barrier: Mhat is complete)
        for (int i = threadIdx.x; i < nrt * nm9; i += nthr) es.Mf[i] = make_float2((float)es.M[i].x, (float)es.M[i].y);
        __syncthreads();
    }

    // ---- row by row, 64-process chunks: chunk c of a row goes to warp (c + rotation of the row) mod GW -- a static deal
    //      that depends on nothing but the row itself, so a row's sums do not depend on how rows were grouped or chunked
    BlkSmem bs;
    bs.meta = es.meta; bs.ph = es.ph; bs.seg = es.seg; bs.M = es.M;
    const double2 *tabA = G.s2 > 0 ? d.evec : d.evecc;
    for (int rt = 0; rt < nrt; rt++) {
        const unsigned *rp = es.rpre + rt * (NU + 1);
        const unsigned total = rp[NU];
        if (total == 0) continue;
        if (MG) {
            int t, lam1; int64_t rold;
            group_row<ORDER>(d, ga, G, rr0 + rt, t, lam1, rold);
            bs.M = const_cast<double2 *>(pre) + (size_t)t * nm9;
        } else bs.M = es.M + rt * nm9;
        const ListEnt *slot = lists + ((size_t)gl * ga.rmaxg + rr0 + rt) * NU * (size_t)capw;
        // the NU slots of the row read as one list: entry i lives in slot w = max{k : rp[k] <= i} at offset i - rp[w]
        auto fetch = [&](unsigned i) -> ListEnt {
            int w = 0;
#pragma unroll
            for (int st = NUMAX >> 1; st > 0; st >>= 1)
                if (st < NU) w += (rp[w + st] <= i) ? st : 0;
            const uint4 v = __ldg(reinterpret_cast<const uint4 *>(slot + (size_t)w * (size_t)capw + (i - rp[w])));
            ListEnt e; e.x = v.x; e.y = v.y; e.w = __hiloint2double((int)v.w, (int)v.z);
            return e;
        };
        double sG = 0.0, sW = 0.0;
        unsigned sC = 0;
        const unsigned first = (unsigned)(warp - (int)es.rot[rt] + nw) % (unsigned)nw;
        for (unsigned base = first * 64; base < total; base += 64 * nw) {
            const bool act0 = base + lane < total, act1 = base + 32 + lane < total;
            const ListEnt e0 = fetch(act0 ? base + lane : base), e1 = fetch(act1 ? base + 32 + lane : base);
            const int qx0 = (int)((e0.x & 0x7fffffffu) >> 6), qx1 = (int)((e1.x & 0x7fffffffu) >> 6);
            const double2 *eA0 = tabA + ((size_t)qx0 * nb + (e0.x & 63u)) * nb;
            const double2 *eA1 = tabA + ((size_t)qx1 * nb + (e1.x & 63u)) * nb;
            const double2 *eB0 = d.evecc + ((size_t)(e0.y >> 6) * nb + (e0.y & 63u)) * nb;
            const double2 *eB1 = d.evecc + ((size_t)(e1.y >> 6) * nb + (e1.y & 63u)) * nb;
            const int3 xc0 = unpack_qc(__ldg(d.qc + qx0)), xc1 = unpack_qc(__ldg(d.qc + qx1));
            double2 V0, V1;
            if constexpr (NAT > 0 && MIX) {
                constexpr int NC = 3 * NAT;
                float2 A0[NC], B0[NC], A1[NC], B1[NC];
                const float2 *tA = G.s2 > 0 ? d.evec32 : d.evecc32;
                const float2 *fA0 = tA + (eA0 - tabA), *fA1 = tA + (eA1 - tabA), *fB0 = d.evecc32 + (eB0 - d.evecc), *fB1 = d.evecc32 + (eB1 - d.evecc);
#pragma unroll
                for (int c = 0; c < NC; c++) { A0[c] = __ldg(fA0 + c); B0[c] = __ldg(fB0 + c); A1[c] = __ldg(fA1 + c); B1[c] = __ldg(fB1 + c); }
                float2 W0, W1;
                contract_process2_f32<NAT>(d, bs, es.Mf + rt * nm9, es.phf, A0, B0, premul(d, xc0), A1, B1, premul(d, xc1), W0, W1);
                V0 = make_double2((double)W0.x, (double)W0.y); V1 = make_double2((double)W1.x, (double)W1.y);
            } else if constexpr (NAT > 0) {
                double2 B0[3 * (NAT > 0 ? NAT : 1)], B1[3 * (NAT > 0 ? NAT : 1)];
                load_evec<3 * NAT>(eB0, B0); load_evec<3 * NAT>(eB1, B1);
                contract_process2<NAT>(d, bs, eA0, B0, premul(d, xc0), eA1, B1, premul(d, xc1), V0, V1);
            } else {
                double2 *As = es.As + (size_t)warp * nb * 64 + lane;   // this lane's two leg-A vectors, [component][process]
                if ((nb & 1) == 0) {
                    for (int c = 0; c < nb; c += 2) {
                        double2 lo, hi;
                        ldg256(eA0 + c, lo, hi); As[c * 64] = lo; As[(c + 1) * 64] = hi;
                        ldg256(eA1 + c, lo, hi); As[c * 64 + 32] = lo; As[(c + 1) * 64 + 32] = hi;
                    }
                } else {
                    for (int c = 0; c < nb; c++) { As[c * 64] = __ldg(eA0 + c); As[c * 64 + 32] = __ldg(eA1 + c); }
                }
                contract_process2_staged(d, bs, As, eB0, premul(d, xc0), eB1, premul(d, xc1), V0, V1);
            }
            if (act0) { sW += e0.w; sG = fma(e0.w, V0.x * V0.x + V0.y * V0.y, sG); sC += 1u + (e0.x >> 31); }
            if (act1) { sW += e1.w; sG = fma(e1.w, V1.x * V1.x + V1.y * V1.y, sG); sC += 1u + (e1.x >> 31); }
        }
        for (int o = 16; o > 0; o >>= 1) {                            // fixed-order warp sums of the row
            sG += __shfl_down_sync(0xffffffffu, sG, o); sW += __shfl_down_sync(0xffffffffu, sW, o);
            sC += __shfl_down_sync(0xffffffffu, sC, o);
        }
        if (lane == 0) { es.accG[warp * ge + rt] = sG; es.accW[warp * ge + rt] = sW; es.accC[warp * ge + rt] = sC; }
    }
    __syncthreads();
    for (int r = threadIdx.x; r < nrt; r += nthr) {
        if (es.rpre[r * (NU + 1) + NU] == 0) continue;
        double tG = 0.0, tW = 0.0;
        unsigned tC = 0;
        for (int w = 0; w < nw; w++) { tG += es.accG[w * ge + r]; tW += es.accW[w * ge + r]; tC += es.accC[w * ge + r]; }
        const double fac = es.rowfac[r];
        partial[es.rold[r]] = make_double2(fac * tG, fac * tW);
        counts[es.rold[r]] = tC;
    }
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------------------------------
// entries one unit of k_enum_g can write for one row: its share of the q_A tiles, every (j_A, j_B) pair admitted
int enum_units(const FpDev &d) {
    const int ntiles = (d.N + 31) >> 5;
    int nu = 1;
    while (2 * nu <= NUMAX && 2 * nu <= ntiles) nu *= 2;
    return nu;
}
int64_t enum_slot_entries(const FpDev &d) {
    const int64_t ntiles = (d.N + 31) >> 5, nu = enum_units(d);
    return (ntiles + nu - 1) / nu * 32 * d.nb * d.nb;
}

cudaError_t launch_enum_g(int order, const FpDev &d, const GroupArgs &ga, int64_t ngc, int64_t capw, ListEnt *lists,
                          uint32_t *wcnt, unsigned int *work, int sm_count, cudaStream_t st) {
    if (ngc <= 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(work, 0, sizeof(unsigned int), st);
    if (e != cudaSuccess) return e;
    const int64_t nunits = ngc * ga.nu;
    const unsigned g = (unsigned)std::min<int64_t>((nunits + GW - 1) / GW, (int64_t)sm_count * FP_ENUM_MINB);
    const bool t6 = d.nb % 6 == 0;
#define FP_ENUM(O, T) k_enum_g<O, T><<<g, GT, 0, st>>>(d, ga, ngc, capw, lists, wcnt, work)
    if (order == 3) { if (t6) FP_ENUM(3, 6); else FP_ENUM(3, 3); }
    else { if (t6) FP_ENUM(4, 6); else FP_ENUM(4, 3); }
#undef FP_ENUM
    return cudaGetLastError();
}

// warps of an evaluator CTA: 4, or -- generic atom count -- as many (at most GEN_WMAX) as the per-warp staging of 64
// leg-A eigenvectors leaves room for beside the tile's tables
static int eval_warps(const FpDev &d, const IfcDev &f, int ge, bool mglobal = false) {
    if (d.nat <= 2) return GW;
    int nw = GEN_WMAX;
    while (nw > 1 && eval_smem_layout(ge, f.nblk, d.L, d.nb, d.nat, enum_units(d), nw, true, false, nullptr, nullptr, mglobal) > 226 * 1024) nw--;
    return nw;
}
size_t eval_smem_bytes(const FpDev &d, const IfcDev &f, int ge, bool mglobal) {   // (with the FP32 copies of the mixed mode)
    return eval_smem_layout(ge, f.nblk, d.L, d.nb, d.nat, enum_units(d), eval_warps(d, f, ge, mglobal), d.nat > 2, d.nat <= 2 && !mglobal,
                            nullptr, nullptr, mglobal);
}

template <int ORDER, int NAT, bool MIX, bool MG = false>
static cudaError_t launch_eval_t(const FpDev &d, const IfcDev &f, const GroupArgs &ga, int64_t ngc, const double2 *pre,
                                 int64_t capw, const ListEnt *lists, const uint32_t *wcnt, int ge, double2 *partial,
                                 uint32_t *counts, cudaStream_t st) {
    const int nw = eval_warps(d, f, ge, MG);
    const size_t smem = eval_smem_layout(ge, f.nblk, d.L, d.nb, d.nat, enum_units(d), nw, NAT == 0, MIX, nullptr, nullptr, MG);
    const int tiles = (ga.rmaxg + ge - 1) / ge;
    const unsigned nthr = 32u * (unsigned)nw;
    static SmemGrant granted;
    cudaError_t e = opt_in_smem(k_eval_g<ORDER, NAT, MIX, MG>, smem, granted);
    if (e != cudaSuccess) return e;
    k_eval_g<ORDER, NAT, MIX, MG><<<(unsigned)(ngc * tiles), nthr, smem, st>>>(d, f, ga, pre, capw, lists, wcnt, ge, tiles, partial, counts);
    return cudaGetLastError();
}

cudaError_t launch_eval_g(int order, const FpDev &d, const IfcDev &f, const GroupArgs &ga, int64_t ngc, const double2 *pre,
                          int64_t capw, const ListEnt *lists, const uint32_t *wcnt, int ge, double2 *partial,
                          uint32_t *counts, bool mixed, bool mglobal, cudaStream_t st) {
    if (ngc <= 0) return cudaSuccess;
#define FP_ARGS d, f, ga, ngc, pre, capw, lists, wcnt, ge, partial, counts, st
    if (order == 3 && mglobal) {                                      // (FP64 only: the mixed mode needs the shared-memory copy)
        if (d.nat == 1) return launch_eval_t<3, 1, false, true>(FP_ARGS);
        if (d.nat == 2) return launch_eval_t<3, 2, false, true>(FP_ARGS);
        return launch_eval_t<3, 0, false, true>(FP_ARGS);
    }
    if (order == 3) {
        if (d.nat == 1) return mixed ? launch_eval_t<3, 1, true>(FP_ARGS) : launch_eval_t<3, 1, false>(FP_ARGS);
        if (d.nat == 2) return mixed ? launch_eval_t<3, 2, true>(FP_ARGS) : launch_eval_t<3, 2, false>(FP_ARGS);
        return launch_eval_t<3, 0, false>(FP_ARGS);
    }
    if (d.nat == 1) return mixed ? launch_eval_t<4, 1, true>(FP_ARGS) : launch_eval_t<4, 1, false>(FP_ARGS);
    if (d.nat == 2) return mixed ? launch_eval_t<4, 2, true>(FP_ARGS) : launch_eval_t<4, 2, false>(FP_ARGS);
    return launch_eval_t<4, 0, false>(FP_ARGS);
#undef FP_ARGS
}
