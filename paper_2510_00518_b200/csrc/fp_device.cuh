// fp_device.cuh -- device helpers shared by the kernels of the CUDA path (fp_kernels.cu, fp_rates.cu).
// Momentum arithmetic modulo the mesh, the pinned broadening / window arithmetic of
// SURVEY.md §8(c) step 3 (compute_sigma PAPER.md:161, filter PAPER.md:163), row decoding, fixed-order block sums.
#pragma once
#include "fp_internal.cuh"

namespace {

// ---------------------------------------------------------------------------------------------------------------------
// helpers
// ---------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ void cfma(double2 &acc, double2 a, double2 b) {   // acc += a*b  (4 DFMA)
    acc.x = fma(a.x, b.x, acc.x);
    acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y);
    acc.y = fma(a.y, b.x, acc.y);
}
__device__ __forceinline__ int3 unpack_qc(int p) { return make_int3(p & 1023, (p >> 10) & 1023, (p >> 20) & 1023); }
__device__ __forceinline__ int wrap(int r, int n) {
    r += (r < 0) ? n : 0;
    r -= (r >= n) ? n : 0;
    return r;
}
// step 1: component-wise modulo; operands are already in [0,N_mu)
__device__ __forceinline__ int3 q_add(const FpDev &d, int3 a, int s, int3 b) {
    return make_int3(wrap(a.x + s * b.x, d.N1), wrap(a.y + s * b.y, d.N2), wrap(a.z + s * b.z, d.N3));
}
__device__ __forceinline__ int q_index(const FpDev &d, int3 c) { return c.x + d.N1 * (c.y + d.N2 * c.z); }
// index into ph1d of phi(q,R): qm = (i1 m1, i2 m2, i3 m3), n = cell offset reduced to [0,N_mu)
__device__ __forceinline__ int phase_idx(const FpDev &d, int3 qm, int n1, int n2, int n3) {
    unsigned x = (unsigned)(qm.x * n1 + qm.y * n2 + qm.z * n3);
    if (d.Lmask >= 0) return (int)(x & (unsigned)d.Lmask);
    // x mod L without a division: floor(x Lmagic / 2^32) with Lmagic = ceil(2^32 / L) is floor(x / L) or one more than
    // that for every 32-bit x, so one conditional correction makes it exact
    const unsigned q = __umulhi(x, d.Lmagic);
    int r = (int)(x - q * (unsigned)d.L);
    return r < 0 ? r + d.L : r;
}
__device__ __forceinline__ int3 premul(const FpDev &d, int3 c) { return make_int3(c.x * d.m1, c.y * d.m2, c.z * d.m3); }

#ifndef FP_LDG256
#define FP_LDG256 1     // gathers of 32-byte aligned records go through one 256-bit load per 32-byte sector (LDG.E.256, sm_100)
#endif
// 32 bytes at a 32-byte aligned address through the read-only path: one request per sector instead of two
__device__ __forceinline__ void ldg256(const void *p, double2 &lo, double2 &hi) {
#if FP_LDG256 && defined(FP_LDG_VOLATILE)
    asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(lo.x), "=d"(lo.y), "=d"(hi.x), "=d"(hi.y) : "l"(p));
#elif FP_LDG256
    asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(lo.x), "=d"(lo.y), "=d"(hi.x), "=d"(hi.y) : "l"(p));
#else
    lo = __ldg(reinterpret_cast<const double2 *>(p)); hi = __ldg(reinterpret_cast<const double2 *>(p) + 1);
#endif
}
__device__ __forceinline__ ModeRec load_rec(const ModeRec *p) {
    double2 a, b;
    ldg256(p, a, b);
    ModeRec r; r.omega = a.x; r.vx = a.y; r.vy = b.x; r.vz = b.y;
    return r;
}
// NC complex components of one eigenvector (NC even: the vector is a whole number of 32-byte sectors)
template <int NC>
__device__ __forceinline__ void load_evec(const double2 *__restrict__ e, double2 *dst) {
    if constexpr (NC % 2 == 0) {
#pragma unroll
        for (int c = 0; c < NC; c += 2) ldg256(e + c, dst[c], dst[c + 1]);
    } else {
#pragma unroll
        for (int c = 0; c < NC; c++) dst[c] = __ldg(e + c);
    }
}

struct Row {
    bool valid;
    int lam, lam1, s1, s2, ch;
    int64_t t;
    int3 qb;          // base q coordinates: q (3ph) or q + s1 q' (4ph)
    double Obase;     // omega (3ph) or fl(omega + s1 omega') (4ph), pinned
};

template <int ORDER>
__device__ __forceinline__ Row make_row(const FpDev &d, const RowArgs &ra, int64_t r) {
    Row row;
    if (ORDER == 3) {
        row.t = r >> 1; row.ch = (int)(r & 1);
        row.lam = ra.targets[row.t]; row.lam1 = -1;
        row.s1 = +1; row.s2 = row.ch == 0 ? +1 : -1;
        double w = d.rec[row.lam].omega;
        row.valid = (w != 0.0);
        row.qb = unpack_qc(d.qc[row.lam / d.nb]);
        row.Obase = w;
    } else {
        int j1 = (int)(r % d.nb); r /= d.nb;
        int qi = (int)(r % ra.nqp); r /= ra.nqp;
        row.ch = (int)(r % 3); row.t = r / 3;
        row.lam = ra.targets[row.t];
        int q1 = ra.qp_begin + qi;
        row.lam1 = q1 * d.nb + j1;
        row.s1 = row.ch == 2 ? -1 : +1; row.s2 = row.ch == 0 ? +1 : -1;
        double w = d.rec[row.lam].omega, w1 = d.rec[row.lam1].omega;
        row.valid = (w != 0.0) && (w1 != 0.0);
        row.qb = q_add(d, unpack_qc(d.qc[row.lam / d.nb]), row.s1, unpack_qc(d.qc[q1]));
        row.Obase = row.s1 > 0 ? __dadd_rn(w, w1) : __dsub_rn(w, w1);
    }
    return row;
}

// compute_sigma(v_A - v_B), in the pinned operation order of SURVEY.md §8(c) step 3 (no FMA contraction)
__device__ __forceinline__ double sigma_pinned(const FpDev &d, const ModeRec &a, const ModeRec &b) {
    if (d.sigma_const > 0.0) return d.sigma_const;
    double dx = __dsub_rn(a.vx, b.vx), dy = __dsub_rn(a.vy, b.vy), dz = __dsub_rn(a.vz, b.vz);
    double t0 = __dadd_rn(__dadd_rn(__dmul_rn(d.B[0], dx), __dmul_rn(d.B[1], dy)), __dmul_rn(d.B[2], dz));
    double t1 = __dadd_rn(__dadd_rn(__dmul_rn(d.B[3], dx), __dmul_rn(d.B[4], dy)), __dmul_rn(d.B[5], dz));
    double t2 = __dadd_rn(__dadd_rn(__dmul_rn(d.B[6], dx), __dmul_rn(d.B[7], dy)), __dmul_rn(d.B[8], dz));
    double s = __dadd_rn(__dadd_rn(__dmul_rn(t0, t0), __dmul_rn(t1, t1)), __dmul_rn(t2, t2));
    return __dmul_rn(d.scale, __dsqrt_rn(__ddiv_rn(s, 6.0)));
}

// Allowed-branch mask of one (qx, ja) pair: bit jb set iff (qx,ja,jb) passes the window (inclusive).
template <int ORDER>
__device__ __forceinline__ uint64_t test_pair(const FpDev &d, const Row &row, int p) {
    ModeRec a = load_rec(d.rec + p);
    if (a.omega == 0.0) return 0;                                   // item 8: zero modes are never a leg
    int qx = p / d.nb;
    int ql = q_index(d, q_add(d, row.qb, row.s2, unpack_qc(d.qc[qx])));
    const ModeRec *rb = d.rec + (size_t)ql * d.nb;
    double base = row.s2 > 0 ? __dadd_rn(row.Obase, a.omega) : __dsub_rn(row.Obase, a.omega);
    uint64_t mask = 0;
    for (int jb = 0; jb < d.nb; jb++) {
        ModeRec b = load_rec(rb + jb);
        if (b.omega == 0.0) continue;
        double sig = sigma_pinned(d, a, b);
        double delta = __dsub_rn(base, b.omega);
        if (sig > 0.0 && fabs(delta) <= __dmul_rn(d.ncut, sig)) mask |= (1ull << jb);
    }
    return mask;
}

// fixed-order block reductions (deterministic: shuffle tree inside a warp, then warp results summed in warp order)
template <typename T>
__device__ __forceinline__ T block_sum(T v, T *sh /* >= 32 */) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
    __syncthreads();
    if (l == 0) sh[w] = v;
    __syncthreads();
    T tot = 0;
    if (threadIdx.x == 0)
        for (int i = 0; i < nw; i++) tot += sh[i];
    return tot;   // valid in thread 0
}


}  // namespace
