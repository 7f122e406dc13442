// fp_contract.cuh -- the per-process (level-2) contraction shared by the fused kernel (fp_rates.cu) and the evaluator of
// the group path (fp_group.cu): compute_Vp of PAPER.md:168,342 in the pre-contracted form of DESIGN.md §5.1,
//   V = sum_b phi(s2 q_A, dR_b) sum_{xy} Mhat_b[x][y] A(atomA_b, x) conj(e~_B(atomB_b, y)).
#pragma once
#include "fp_device.cuh"

namespace {

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
// complex MACs, and the two dependency chains interleave (NAT > 0 only).  The conj(e~_B) vectors of both processes are
// resident (B0, B1); the three leg-A components of an atom are loaded when that atom's blocks start (72 instead of 96
// registers of eigenvector state: at the 168-register cap of three CTAs per SM the compiler otherwise serialises
// independent DFMA chains -- measured 676 -> 651 ms per config-3 step, and 630 with the t-step written row by row of
// Mhat).  Block order as everywhere else:
// (atomA, atomB, dR).
template <int NAT>
__device__ __forceinline__ void contract_process2(const FpDev &d, const BlkSmem &bs, const double2 *__restrict__ eA0, const double2 *B0,
                                                  int3 q0, const double2 *__restrict__ eA1, const double2 *B1, int3 q1, double2 &V0,
                                                  double2 &V1) {
    V0 = make_double2(0.0, 0.0); V1 = make_double2(0.0, 0.0);
#pragma unroll
    for (int a = 0; a < NAT; a++) {
        double2 A0[3], A1[3];
#pragma unroll
        for (int x = 0; x < 3; x++) { A0[x] = __ldg(eA0 + 3 * a + x); A1[x] = __ldg(eA1 + 3 * a + x); }
#pragma unroll
        for (int c = 0; c < NAT; c++) {
            const int b1 = bs.seg[a * NAT + c + 1];
            for (int b = bs.seg[a * NAT + c]; b < b1; b++) {
                const int4 m = bs.meta[b];
                const double2 p0 = bs.ph[phase_idx(d, q0, m.y, m.z, m.w)], p1 = bs.ph[phase_idx(d, q1, m.y, m.z, m.w)];
                const double2 *M = bs.M + 9 * b;
                double2 u0 = make_double2(0.0, 0.0), u1 = make_double2(0.0, 0.0);
                double2 t0[3], t1[3];                                 // t[y] = sum_x Mhat[x][y] A[x], row by row of Mhat: the six
#pragma unroll                                                        // t's of the two processes are twelve independent DFMA chains
                for (int y = 0; y < 3; y++) { t0[y] = make_double2(0.0, 0.0); t1[y] = make_double2(0.0, 0.0); }
#pragma unroll
                for (int x = 0; x < 3; x++)
#pragma unroll
                    for (int y = 0; y < 3; y++) {
                        const double2 mm = M[3 * x + y];
                        cfma(t0[y], mm, A0[x]); cfma(t1[y], mm, A1[x]);
                    }
#pragma unroll
                for (int y = 0; y < 3; y++) { cfma(u0, t0[y], B0[3 * c + y]); cfma(u1, t1[y], B1[3 * c + y]); }
                cfma(V0, u0, p0); cfma(V1, u1, p1);
            }
        }
    }
}

// Mixed precision (fp_set_precision): the same two-process contraction in FP32 -- Mhat, phases and both
// eigenvectors rounded to FP32, FP32 FMAs.  NAT > 0 only.
__device__ __forceinline__ void cfmaf(float2 &acc, float2 a, float2 b) {
    acc.x = fmaf(a.x, b.x, acc.x);
    acc.x = fmaf(-a.y, b.y, acc.x);
    acc.y = fmaf(a.x, b.y, acc.y);
    acc.y = fmaf(a.y, b.x, acc.y);
}
template <int NAT>
__device__ __forceinline__ void contract_process2_f32(const FpDev &d, const BlkSmem &bs, const float2 *Mf, const float2 *phf,
                                                      const float2 *A0, const float2 *B0, int3 q0, const float2 *A1,
                                                      const float2 *B1, int3 q1, float2 &V0, float2 &V1) {
    V0 = make_float2(0.f, 0.f); V1 = make_float2(0.f, 0.f);
#pragma unroll
    for (int a = 0; a < NAT; a++)
#pragma unroll
        for (int c = 0; c < NAT; c++) {
            const int b1 = bs.seg[a * NAT + c + 1];
            for (int b = bs.seg[a * NAT + c]; b < b1; b++) {
                const int4 m = bs.meta[b];
                const float2 p0 = phf[phase_idx(d, q0, m.y, m.z, m.w)], p1 = phf[phase_idx(d, q1, m.y, m.z, m.w)];
                const float2 *M = Mf + 9 * b;
                float2 u0 = make_float2(0.f, 0.f), u1 = make_float2(0.f, 0.f);
#pragma unroll
                for (int y = 0; y < 3; y++) {
                    float2 t0 = make_float2(0.f, 0.f), t1 = make_float2(0.f, 0.f);
#pragma unroll
                    for (int x = 0; x < 3; x++) {
                        const float2 mm = M[3 * x + y];
                        cfmaf(t0, mm, A0[3 * a + x]); cfmaf(t1, mm, A1[3 * a + x]);
                    }
                    cfmaf(u0, t0, B0[3 * c + y]); cfmaf(u1, t1, B1[3 * c + y]);
                }
                cfmaf(V0, u0, p0); cfmaf(V1, u1, p1);
            }
        }
}

// The same for any atom count, every eigenvector component fetched once: the leg-A vectors of the two processes are
// staged by the caller in shared memory (As[comp * 64 + 32 h], already offset by the lane: each lane reads back only
// what it wrote), the loop runs atom-B-major with the three conj(e~_B) components of atom c in registers, and the sum
// over y is taken once per atom c:
//   W_c[y] = sum_{b : atomB_b = c} phi_b sum_x Mhat_b[x][y] A(atomA_b, x),   V = sum_c sum_y W_c[y] conj(e~_B(c, y))
// -- 12 complex MACs per block and process plus 3 per atom c.  Blocks are sorted by (atomA, atomB): seg[a nat + c].
__device__ __forceinline__ void contract_process2_staged(const FpDev &d, const BlkSmem &bs, const double2 *As,
                                                         const double2 *__restrict__ eB0, int3 q0,
                                                         const double2 *__restrict__ eB1, int3 q1, double2 &V0, double2 &V1) {
    V0 = make_double2(0.0, 0.0); V1 = make_double2(0.0, 0.0);
    const int nat = d.nat;
    for (int c = 0; c < nat; c++) {
        double2 B0[3], B1[3], W0[3], W1[3];
#pragma unroll
        for (int y = 0; y < 3; y++) {
            B0[y] = __ldg(eB0 + 3 * c + y); B1[y] = __ldg(eB1 + 3 * c + y);   // (first needed after all blocks of atom c)
            W0[y] = make_double2(0.0, 0.0); W1[y] = make_double2(0.0, 0.0);
        }
        for (int a = 0; a < nat; a++) {
            const int b0 = bs.seg[a * nat + c], b1 = bs.seg[a * nat + c + 1];
            if (b0 == b1) continue;
            double2 A0[3], A1[3];
#pragma unroll
            for (int x = 0; x < 3; x++) { A0[x] = As[(3 * a + x) * 64]; A1[x] = As[(3 * a + x) * 64 + 32]; }
#pragma unroll 2                                                      // (measured on B200, config 4: 1 / 2 / 3 / 4 -> 3180 / 3091 / 3183 / 3208 ms)
            for (int b = b0; b < b1; b++) {
                const int4 m = bs.meta[b];
                const double2 p0 = bs.ph[phase_idx(d, q0, m.y, m.z, m.w)], p1 = bs.ph[phase_idx(d, q1, m.y, m.z, m.w)];
                const double2 *M = bs.M + 9 * b;
#pragma unroll
                for (int y = 0; y < 3; y++) {
                    double2 t0 = make_double2(0.0, 0.0), t1 = make_double2(0.0, 0.0);
#pragma unroll
                    for (int x = 0; x < 3; x++) {
                        const double2 mm = M[3 * x + y];
                        cfma(t0, mm, A0[x]); cfma(t1, mm, A1[x]);
                    }
                    cfma(W0[y], t0, p0); cfma(W1[y], t1, p1);
                }
            }
        }
#pragma unroll
        for (int y = 0; y < 3; y++) { cfma(V0, W0[y], B0[y]); cfma(V1, W1[y], B1[y]); }
    }
}

}  // namespace
