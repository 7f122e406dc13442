// fp_host.cu -- host side of the C ABI (include/fourphonon.h): argument checking, IFC block analysis, workspace
// carving, the bounded-memory loop over super-chunks of targets (Algorithm 5) and launches.
// All arithmetic of the method runs in the kernels of fp_kernels.cu; the only floating-point work here is the 3x3
// reciprocal-lattice setup B_mu = b_mu/N_mu in the pinned order of SURVEY.md §8(c) step 3 and the unit constants.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <tuple>

#include "fp_internal.cuh"

#ifndef FP_SLOT_DIV
#define FP_SLOT_DIV 4        // list slot = 1/FP_SLOT_DIV of the candidates a warp can meet
#endif
#ifndef FP_EVAL_TILE_BYTES
#define FP_EVAL_TILE_BYTES (16 * 1024)   // Mhat tables of the rows of one evaluator tile (k_eval_g)
#endif

namespace {

// ---- unit constants (SURVEY.md §8(c) "Constants"), derived from CODATA 2018 ------------------------------------------
constexpr double kHbar = 1.054571817e-34;     // J s
constexpr double kKb = 1.380649e-23;          // J/K
constexpr double kQe = 1.602176634e-19;       // C
constexpr double kAmu = 1.66053906660e-27;    // kg
const double kPi = 3.141592653589793238462643383279502884;

double hbar_over_kb() { return kHbar / kKb * 1e12; }                                  // ps K
double const_c3() {                                                                    // (pi hbar/4)(eV/A^3)^2/u^3/(rad/ps)^4 in 1/ps
    double f = kQe * 1e30;
    return kPi * kHbar * 0.25 * f * f / (kAmu * kAmu * kAmu) * 1e-60;
}
double const_c4() {                                                                    // (pi hbar^2/8)(eV/A^4)^2/u^4/(rad/ps)^5 in 1/ps
    double f = kQe * 1e40;
    return kPi * kHbar * kHbar * 0.125 * f * f / (kAmu * kAmu * kAmu * kAmu) * 1e-72;
}
double const_ckappa() { return kHbar * kHbar / kKb * 1e46; }                           // W/(m K) per unit

thread_local std::string g_setup_err;

int fail(fp_ctx *ctx, int code, const std::string &msg) {
    if (ctx) ctx->err = msg; else g_setup_err = msg;
    return code;
}
#define CU(call)                                                                                         \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess)                                                                           \
            return fail(ctx, FP_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));              \
    } while (0)

size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

struct Bump {
    char *base; size_t off, end;
    template <typename T> T *take(size_t n) {
        size_t o = align_up(off);
        size_t b = n * sizeof(T);
        if (o + b > end) return nullptr;
        off = o + b;
        return reinterpret_cast<T *>(base + o);
    }
};

int imod(long a, int n) { long r = a % n; return (int)(r < 0 ? r + n : r); }
long gcdl(long a, long b) { while (b) { long t = a % b; a = b; b = t; } return a; }

// Host-side analysis of an IFC list: group clusters into contraction blocks (atomA, atomB, dR) -- DESIGN.md §5.
struct IfcHost {
    int n = 0, nblk = 0, ncomp = 0;
    std::vector<int4> meta0, meta1, blk_meta;
    std::vector<double> phi;
    std::vector<int> blk_start, seg;
};

int analyse_ifc(const fp_ifc *f, int order, int nat, const int32_t mesh[3], IfcHost &h, std::string &err) {
    const int ncomp = order == 3 ? 27 : 81;
    h.n = (int)f->n; h.ncomp = ncomp;
    if (f->n < 0 || f->n > (1 << 24)) { err = "IFC list size out of range"; return FP_EINVAL; }
    if (f->n > 0 && (!f->atoms || !f->cells || !f->phi)) { err = "IFC list has null arrays"; return FP_EINVAL; }
    typedef std::tuple<int, int, int, int, int> Key;       // atomA, atomB, d1, d2, d3
    std::map<Key, int> blocks;
    std::vector<Key> key(h.n);
    for (int c = 0; c < h.n; c++) {
        const int32_t *at = f->atoms + (size_t)c * order;
        for (int m = 0; m < order; m++)
            if (at[m] < 0 || at[m] >= nat) { err = "IFC atom index out of range"; return FP_EINVAL; }
        const int32_t *RA = f->cells + (size_t)c * (order - 1) * 3 + (order - 3) * 3;   // leg A: j (3ph) / k (4ph)
        const int32_t *RB = RA + 3;                                                      // leg B: k (3ph) / l (4ph)
        key[c] = Key(at[order - 2], at[order - 1], imod((long)RA[0] - RB[0], mesh[0]), imod((long)RA[1] - RB[1], mesh[1]),
                     imod((long)RA[2] - RB[2], mesh[2]));
        blocks.emplace(key[c], 0);
    }
    h.nblk = (int)blocks.size();
    int id = 0;
    h.blk_meta.resize(h.nblk);
    h.seg.assign(nat * nat + 1, 0);
    for (auto &kv : blocks) {                                // std::map iterates sorted by (atomA, atomB, dR)
        kv.second = id;
        const Key &k = kv.first;
        h.blk_meta[id] = make_int4(std::get<0>(k) | (std::get<1>(k) << 16), std::get<2>(k), std::get<3>(k),
                                   std::get<4>(k));           // {atomA | atomB << 16, dR}; key order = sort order
        h.seg[std::get<0>(k) * nat + std::get<1>(k) + 1]++;
        id++;
    }
    for (int i = 0; i < nat * nat; i++) h.seg[i + 1] += h.seg[i];
    std::vector<int> order_idx(h.n);
    for (int c = 0; c < h.n; c++) order_idx[c] = c;
    std::stable_sort(order_idx.begin(), order_idx.end(), [&](int a, int b) { return blocks[key[a]] < blocks[key[b]]; });
    h.blk_start.assign(h.nblk + 1, 0);
    h.meta0.resize(h.n); h.meta1.resize(h.n); h.phi.resize((size_t)h.n * ncomp);
    for (int s = 0; s < h.n; s++) {
        int c = order_idx[s];
        const int32_t *at = f->atoms + (size_t)c * order;
        const int32_t *cl = f->cells + (size_t)c * (order - 1) * 3;
        const int32_t *RL = cl + (order - 2) * 3;            // last leg: k (3ph) / l (4ph)
        h.blk_start[blocks[key[c]] + 1]++;
        h.meta0[s] = make_int4(at[0], imod(RL[0], mesh[0]), imod(RL[1], mesh[1]), imod(RL[2], mesh[2]));
        if (order == 4)                                      // level 1: atom j and Rj - Rl
            h.meta1[s] = make_int4(at[1], imod((long)cl[0] - RL[0], mesh[0]), imod((long)cl[1] - RL[1], mesh[1]),
                                   imod((long)cl[2] - RL[2], mesh[2]));
        else
            h.meta1[s] = make_int4(0, 0, 0, 0);
        std::memcpy(&h.phi[(size_t)s * ncomp], f->phi + (size_t)c * ncomp, sizeof(double) * ncomp);
    }
    for (int b = 0; b < h.nblk; b++) h.blk_start[b + 1] += h.blk_start[b];
    return FP_OK;
}

// Is the IFC list invariant under the exchange of its last two legs -- Phi^{abgt}(i,j,k Rk,l Rl) = Phi^{abtg}(i,j,l Rl,k Rk)
// for order 4, Phi^{abg}(i,j Rj,k Rk) = Phi^{agb}(i,k Rk,j Rj) for order 3 (a derivative symmetry every physical
// force-constant set has)?  Then |V| and the weights of the channels whose two free legs are both conjugated (3ph -,
// 4ph +- and --) are symmetric under the exchange of those legs and the split path evaluates
// each unordered pair once.  Tolerance: 1e-13 of the largest entry.
bool ifc_last_legs_symmetric(const fp_ifc *f, int order) {
    typedef std::vector<int> K;                              // fixed legs, then the two exchangeable legs (atom, R)
    const int nfix = order - 3;                              // order 4: leg j is fixed
    const int ncomp = order == 3 ? 27 : 81, nlead = ncomp / 9;
    std::map<K, int64_t> idx;
    auto key = [&](int64_t c, bool swap) {
        const int32_t *at = f->atoms + c * order, *cl = f->cells + c * (order - 1) * 3;
        K k;
        k.push_back(at[0]);
        for (int m = 0; m < nfix; m++) { k.push_back(at[1 + m]); for (int x = 0; x < 3; x++) k.push_back(cl[3 * m + x]); }
        const int a = order - 2, b = order - 1;              // the last two legs
        const int32_t *Ra = cl + 3 * (a - 1), *Rb = cl + 3 * (b - 1);
        const int la = swap ? b : a, lb = swap ? a : b;
        const int32_t *R1 = swap ? Rb : Ra, *R2 = swap ? Ra : Rb;
        k.push_back(at[la]); for (int x = 0; x < 3; x++) k.push_back(R1[x]);
        k.push_back(at[lb]); for (int x = 0; x < 3; x++) k.push_back(R2[x]);
        return k;
    };
    double big = 0.0;
    for (int64_t c = 0; c < f->n; c++) {
        if (!idx.emplace(key(c, false), c).second) return false;   // duplicate cluster: do not reason about sums, stay safe
        for (int x = 0; x < ncomp; x++) big = std::max(big, std::fabs(f->phi[c * ncomp + x]));
    }
    const double tol = 1e-13 * big;
    for (int64_t c = 0; c < f->n; c++) {
        auto it = idx.find(key(c, true));
        const double *P = f->phi + c * ncomp;
        if (it == idx.end()) {                                // no partner: symmetric only if the cluster is zero
            for (int x = 0; x < ncomp; x++) if (std::fabs(P[x]) > tol) return false;
            continue;
        }
        const double *Q = f->phi + it->second * ncomp;
        for (int ab = 0; ab < nlead; ab++)
            for (int g = 0; g < 3; g++)
                for (int t = 0; t < 3; t++)
                    if (std::fabs(P[ab * 9 + g * 3 + t] - Q[ab * 9 + t * 3 + g]) > tol) return false;
    }
    return true;
}

size_t ifc_resident_bytes(int64_t n, int order, int nat) {
    size_t ncomp = order == 3 ? 27 : 81;
    size_t b = 0;
    b += align_up(n * sizeof(int4)) * 2 + align_up(n * ncomp * sizeof(double));
    b += align_up((n + 1) * sizeof(int)) + align_up(n * sizeof(int4)) + align_up((nat * nat + 1) * sizeof(int));
    return b + 256 * 8;
}

size_t tables_resident_bytes(int nat, const int32_t mesh[3], long L) {
    size_t N = (size_t)mesh[0] * mesh[1] * mesh[2], nb = 3 * (size_t)nat, M = N * nb;
    return align_up(M * sizeof(ModeRec)) + align_up(M * 16) * 2 + align_up(M * 8) * 2 + align_up(M * nb * 16) * 2 + align_up(M * nb * 8) * 2 +
           align_up((size_t)L * 16) + align_up(N * 4) + align_up(N * 8) + align_up(nat * 8) + 256 * 12;
}

long mesh_lcm(const int32_t mesh[3]) {
    long L = mesh[0];
    L = L / gcdl(L, mesh[1]) * mesh[1];
    L = L / gcdl(L, mesh[2]) * mesh[2];
    return L;
}

int upload_ifc(fp_ctx *ctx, Bump &bump, const IfcHost &h, IfcDev &dv, cudaStream_t st) {
    int nat = ctx->d.nat;
    int4 *m0 = bump.take<int4>(std::max(h.n, 1));
    int4 *m1 = bump.take<int4>(std::max(h.n, 1));
    double *phi = bump.take<double>(std::max<size_t>((size_t)h.n * h.ncomp, 1));
    int *bs = bump.take<int>(h.nblk + 1);
    int4 *bm = bump.take<int4>(std::max(h.nblk, 1));
    int *seg = bump.take<int>(nat * nat + 1);
    if (!m0 || !m1 || !phi || !bs || !bm || !seg) return fail(ctx, FP_ENOMEM, "workspace too small for IFC tables");
    if (h.n > 0) {
        CU(cudaMemcpyAsync(m0, h.meta0.data(), h.n * sizeof(int4), cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(m1, h.meta1.data(), h.n * sizeof(int4), cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(phi, h.phi.data(), h.phi.size() * sizeof(double), cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(bm, h.blk_meta.data(), h.nblk * sizeof(int4), cudaMemcpyHostToDevice, st));
    }
    CU(cudaMemcpyAsync(bs, h.blk_start.data(), (h.nblk + 1) * sizeof(int), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(seg, h.seg.data(), (nat * nat + 1) * sizeof(int), cudaMemcpyHostToDevice, st));
    CU(cudaStreamSynchronize(st));                                   // host vectors go out of scope after setup
    dv.n = h.n; dv.nblk = h.nblk; dv.ncomp = h.ncomp;
    dv.cl_meta0 = m0; dv.cl_meta1 = m1; dv.phi = phi; dv.blk_start = bs; dv.blk_meta = bm; dv.seg = seg;
    return FP_OK;
}

// ---- profiling ----------------------------------------------------------------------------------------------------------
struct ProfScope {
    fp_ctx *ctx; cudaStream_t st; int idx = -1;
    ProfScope(fp_ctx *c, int cat, cudaStream_t s) : ctx(c), st(s) {
        if (!ctx->profiling) return;
        EventRec r; r.cat = cat;
        cudaEvent_t *ev[2] = {&r.a, &r.b};
        for (auto e : ev) {                                           // events are pooled across fp_profile_reset
            if (!ctx->pool.empty()) { *e = ctx->pool.back(); ctx->pool.pop_back(); }
            else if (cudaEventCreate(e) != cudaSuccess) return;
        }
        cudaEventRecord(r.a, st);
        ctx->events.push_back(r);
        idx = (int)ctx->events.size() - 1;
    }
    ~ProfScope() { if (idx >= 0) cudaEventRecord(ctx->events[idx].b, st); }
};

}  // namespace

// =========================================================================================================================
// public ABI
// =========================================================================================================================
extern "C" {

const char *fp_version(void) { return "fourphonon-b200 0.1 (sm_100a)"; }

void fp_constants(double out[4]) { out[0] = const_c3(); out[1] = const_c4(); out[2] = const_ckappa(); out[3] = hbar_over_kb(); }

const char *fp_last_error(const fp_ctx *ctx) { return ctx ? ctx->err.c_str() : g_setup_err.c_str(); }

size_t fp_workspace_bytes(const fp_crystal *crystal, const int32_t mesh[3], const fp_ifc *ifc3, const fp_ifc *ifc4,
                          size_t scratch_bytes) {
    if (!crystal || !mesh || crystal->natoms <= 0 || mesh[0] <= 0 || mesh[1] <= 0 || mesh[2] <= 0) return 0;
    size_t b = tables_resident_bytes(crystal->natoms, mesh, mesh_lcm(mesh));
    if (ifc3) b += ifc_resident_bytes(ifc3->n, 3, crystal->natoms);
    if (ifc4) b += ifc_resident_bytes(ifc4->n, 4, crystal->natoms);
    // staging of the raw mode arrays during fp_setup lives in the scratch region
    size_t N = (size_t)mesh[0] * mesh[1] * mesh[2], nb = 3 * (size_t)crystal->natoms;
    size_t staging = align_up(N * nb * 8) + align_up(N * nb * nb * 16) + align_up(N * nb * 24) + 1024;
    return b + std::max(scratch_bytes, staging) + 4096;
}

int fp_setup(const fp_crystal *crystal, const double *masses, const double *omega, const double *eig, const double *vg,
             fp_memloc loc, const fp_ifc *ifc3, const fp_ifc *ifc4, const int32_t mesh[3], double T,
             const fp_broadening *br, void *workspace, size_t workspace_bytes, void *stream, fp_ctx **out) {
    fp_ctx *ctx = nullptr;                                            // errors before allocation go to g_setup_err
    if (!out) return fail(ctx, FP_EINVAL, "out is null");
    *out = nullptr;
    if (!crystal || !masses || !omega || !eig || !vg || !mesh || !br || !workspace)
        return fail(ctx, FP_EINVAL, "null argument");
    const int nat = crystal->natoms;
    if (nat <= 0 || 3 * nat > FP_MAX_NB) return fail(ctx, FP_EINVAL, "natoms must be in [1,21]");
    for (int m = 0; m < 3; m++)
        if (mesh[m] <= 0 || mesh[m] > 1024) return fail(ctx, FP_EINVAL, "mesh dimensions must be in [1,1024]");
    if (!(T > 0.0)) return fail(ctx, FP_EINVAL, "T must be > 0");
    if (!(br->scale > 0.0)) return fail(ctx, FP_EINVAL, "broadening scale must be > 0");
    if (!(br->ncut >= 0.0)) return fail(ctx, FP_EINVAL, "ncut must be >= 0");
    if (!(br->sigma_const >= 0.0)) return fail(ctx, FP_EINVAL, "sigma_const must be >= 0");
    for (int a = 0; a < nat; a++)
        if (!(masses[a] > 0.0)) return fail(ctx, FP_EINVAL, "masses must be > 0");
    const long L = mesh_lcm(mesh);
    if (L > FP_MAX_L) return fail(ctx, FP_EINVAL, "lcm of the mesh dimensions exceeds 4096");
    const size_t N = (size_t)mesh[0] * mesh[1] * mesh[2], nb = 3 * (size_t)nat, M = N * nb;
    if (M * nb > (size_t)1 << 31 || N > (size_t)1 << 20)
        return fail(ctx, FP_EINVAL, "more than 2^20 q-points (32-bit candidate codes)");
    if ((reinterpret_cast<uintptr_t>(workspace) & 255) != 0) return fail(ctx, FP_EINVAL, "workspace must be 256-byte aligned");

    IfcHost h3, h4;
    std::string err;
    if (ifc3) { int rc = analyse_ifc(ifc3, 3, nat, mesh, h3, err); if (rc) return fail(ctx, rc, err); }
    if (ifc4) { int rc = analyse_ifc(ifc4, 4, nat, mesh, h4, err); if (rc) return fail(ctx, rc, err); }

    ctx = new fp_ctx();
    cudaStream_t st = (cudaStream_t)stream;
    auto bail = [&](int code) { g_setup_err = ctx->err; delete ctx; return code; };
#undef CU
#define CU(call)                                                                                         \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess) {                                                                         \
            fail(ctx, FP_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));                     \
            return bail(FP_ECUDA);                                                                       \
        }                                                                                                \
    } while (0)

    int dev = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, dev));
    ctx->ws = (char *)workspace; ctx->ws_bytes = workspace_bytes;
    ctx->device = dev;

    FpDev &d = ctx->d;
    d.nat = nat; d.nb = (int)nb; d.N = (int)N; d.N1 = mesh[0]; d.N2 = mesh[1]; d.N3 = mesh[2];
    d.L = (int)L; d.m1 = (int)(L / mesh[0]); d.m2 = (int)(L / mesh[1]); d.m3 = (int)(L / mesh[2]);
    d.Lmask = (L & (L - 1)) == 0 ? (int)(L - 1) : -1;
    d.Lmagic = (unsigned)((((unsigned long long)1 << 32) + (unsigned long long)L - 1) / (unsigned long long)L);
    d.scale = br->scale; d.ncut = br->ncut; d.sigma_const = br->sigma_const; d.T = T;
    {   // B_mu = b_mu/N_mu, pinned order; host code is compiled with -ffp-contract=off
        const double *a1 = crystal->lattvec, *a2 = a1 + 3, *a3 = a1 + 6;
        double c1[3], c2[3], c3[3];
        c1[0] = (a2[1] * a3[2]) - (a2[2] * a3[1]); c1[1] = (a2[2] * a3[0]) - (a2[0] * a3[2]); c1[2] = (a2[0] * a3[1]) - (a2[1] * a3[0]);
        c2[0] = (a3[1] * a1[2]) - (a3[2] * a1[1]); c2[1] = (a3[2] * a1[0]) - (a3[0] * a1[2]); c2[2] = (a3[0] * a1[1]) - (a3[1] * a1[0]);
        c3[0] = (a1[1] * a2[2]) - (a1[2] * a2[1]); c3[1] = (a1[2] * a2[0]) - (a1[0] * a2[2]); c3[2] = (a1[0] * a2[1]) - (a1[1] * a2[0]);
        volatile double vol = (a1[0] * c1[0] + a1[1] * c1[1]) + a1[2] * c1[2];
        if (!(std::fabs(vol) > 0.0)) { fail(ctx, FP_EINVAL, "lattice vectors are singular"); return bail(FP_EINVAL); }
        const double twopi = 2.0 * 3.14159265358979323846;
        for (int x = 0; x < 3; x++) {
            d.B[0 + x] = ((twopi * c1[x]) / vol) / (double)mesh[0];
            d.B[3 + x] = ((twopi * c2[x]) / vol) / (double)mesh[1];
            d.B[6 + x] = ((twopi * c3[x]) / vol) / (double)mesh[2];
        }
        ctx->vol = std::fabs(vol);
    }

    // ---- carve resident tables -----------------------------------------------------------------------------------
    Bump bump{ctx->ws, 0, workspace_bytes};
    ModeRec *rec = bump.take<ModeRec>(M);
    float4 *recf = bump.take<float4>(M);
    float2 *recn = bump.take<float2>(M);
    unsigned long long *maxima = bump.take<unsigned long long>(2);
    double *occ = bump.take<double>(M);
    double2 *aux = bump.take<double2>(M);
    double2 *evec = bump.take<double2>(M * nb);
    double2 *evecc = bump.take<double2>(M * nb);
    float2 *evec32 = bump.take<float2>(M * nb), *evecc32 = bump.take<float2>(M * nb);
    double2 *ph1d = bump.take<double2>(L);
    int *qc = bump.take<int>(N);
    float2 *qmm = bump.take<float2>(N);
    double *masses_dev = bump.take<double>(nat);
    if (!rec || !recf || !recn || !maxima || !occ || !aux || !evec || !evecc || !evec32 || !evecc32 || !ph1d || !qc || !qmm || !masses_dev) {
        fail(ctx, FP_ENOMEM, "workspace too small for the mode tables"); return bail(FP_ENOMEM);
    }
    d.rec = rec; d.recf = recf; d.recn = recn; d.occ = occ; d.aux = aux; d.evec = evec; d.evecc = evecc; d.evec32 = evec32; d.evecc32 = evecc32; d.ph1d = ph1d; d.qc = qc; d.qmm = qmm;
    // executed FP64 flops per matrix element: 13 complex MACs per block (nat <= 2: contract_process2); generic
    // atom count (contract_process2_staged): 12 per block + 3 per atom B that has blocks; 8 flop per complex MAC
    auto flops_elem = [&](const IfcHost &h) {
        if (nat <= 2) return 8.0 * 13.0 * h.nblk;
        int nc = 0;
        for (int c = 0; c < nat; c++) {
            bool any = false;
            for (int a = 0; a < nat; a++) any = any || h.seg[a * nat + c + 1] > h.seg[a * nat + c];
            nc += any ? 1 : 0;
        }
        return 8.0 * (12.0 * h.nblk + 3.0 * nc);
    };
    if (ifc3) ctx->flops_elem3 = flops_elem(h3);
    if (ifc4) ctx->flops_elem4 = flops_elem(h4);
    if (ifc3) {
        int rc = upload_ifc(ctx, bump, h3, ctx->i3, st); if (rc) return bail(rc);
        ctx->has3 = true;
        ctx->sym23 = ifc_last_legs_symmetric(ifc3, 3);
    }
    if (ifc4) {
        int rc = upload_ifc(ctx, bump, h4, ctx->i4, st); if (rc) return bail(rc);
        ctx->has4 = true;
        ctx->sym34 = ifc_last_legs_symmetric(ifc4, 4);
    }
    ctx->resident = align_up(bump.off);

    // ---- stage raw mode arrays (scratch region) and validate omega on the host ---------------------------------------
    const double *d_omega = omega, *d_eig = eig, *d_vg = vg;
    std::vector<double> h_omega(M);
    if (loc == FP_MEM_HOST) {
        Bump sc{ctx->ws, ctx->resident, workspace_bytes};
        double *so = sc.take<double>(M), *se = sc.take<double>(M * nb * 2), *sv = sc.take<double>(M * 3);
        if (!so || !se || !sv) { fail(ctx, FP_ENOMEM, "workspace too small to stage the mode arrays"); return bail(FP_ENOMEM); }
        CU(cudaMemcpyAsync(so, omega, M * 8, cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(se, eig, M * nb * 16, cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(sv, vg, M * 24, cudaMemcpyHostToDevice, st));
        d_omega = so; d_eig = se; d_vg = sv;
        std::memcpy(h_omega.data(), omega, M * 8);
    } else {
        CU(cudaMemcpyAsync(h_omega.data(), omega, M * 8, cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
    }
    double wmax = 0.0, wmin = INFINITY;
    for (size_t m = 0; m < M; m++) {
        double w = h_omega[m];
        if (!(w >= 0.0) || !std::isfinite(w)) { fail(ctx, FP_EINVAL, "omega has a NaN, infinite or negative entry"); return bail(FP_EINVAL); }
        wmax = std::max(wmax, w);
        if (w > 0.0) wmin = std::min(wmin, w);
    }
    d.wmax = wmax; d.wmin = std::min(wmin, wmax);
    for (size_t m = 0; m < M; m++)
        if (h_omega[m] > 0.0 && h_omega[m] < 1e-6 * wmax) {
            fail(ctx, FP_EINVAL, "omega has a near-zero entry (0 < omega < 1e-6*omega_max); zero modes must be exactly 0");
            return bail(FP_EINVAL);
        }
    {   // time-reversal check of the mode arrays (bitwise: the window decision, hence the counts, must map exactly)
        std::vector<double> h_eig, h_vg;
        const double *he = eig, *hv = vg;
        if (loc != FP_MEM_HOST) {
            h_eig.resize(M * nb * 2); h_vg.resize(M * 3);
            CU(cudaMemcpyAsync(h_eig.data(), eig, M * nb * 16, cudaMemcpyDeviceToHost, st));
            CU(cudaMemcpyAsync(h_vg.data(), vg, M * 24, cudaMemcpyDeviceToHost, st));
            CU(cudaStreamSynchronize(st));
            he = h_eig.data(); hv = h_vg.data();
        }
        ctx->qpartner.resize(N);
        bool ok = true;
        for (int i3 = 0; i3 < mesh[2]; i3++)
            for (int i2 = 0; i2 < mesh[1]; i2++)
                for (int i1 = 0; i1 < mesh[0]; i1++) {
                    const size_t iq = i1 + (size_t)mesh[0] * (i2 + (size_t)mesh[1] * i3);
                    const size_t ip = (size_t)((mesh[0] - i1) % mesh[0]) +
                                      (size_t)mesh[0] * (((mesh[1] - i2) % mesh[1]) + (size_t)mesh[1] * ((mesh[2] - i3) % mesh[2]));
                    ctx->qpartner[iq] = (int32_t)ip;
                    if (!ok || ip <= iq) continue;                    // each pair once; a self-conjugate q-point needs nothing
                    for (size_t j = 0; j < nb && ok; j++) {
                        const size_t a = iq * nb + j, b = ip * nb + j;
                        ok = h_omega[a] == h_omega[b] && hv[3 * a] == -hv[3 * b] && hv[3 * a + 1] == -hv[3 * b + 1] &&
                             hv[3 * a + 2] == -hv[3 * b + 2];
                        for (size_t c = 0; c < nb && ok; c++)
                            ok = he[2 * (a * nb + c)] == he[2 * (b * nb + c)] && he[2 * (a * nb + c) + 1] == -he[2 * (b * nb + c) + 1];
                    }
                }
        ctx->trs_ok = ok;
    }
    CU(cudaMemcpyAsync(masses_dev, masses, nat * 8, cudaMemcpyHostToDevice, st));
    // stage 1 of the FP32 pre-filter: |Delta_f| <= n'_a + n'_b with n' = cs |u| (1+1e-6) + slack
    d.pfCs = d.sigma_const > 0.0 ? 0.5 * d.ncut * d.sigma_const : d.ncut * d.scale / std::sqrt(6.0);
    d.pfSlack = 2e-6 * wmax;                                          // per leg; covers |Delta_f - Delta| and 4 FP32 adds
    launch_tables(d, d_omega, d_eig, d_vg, masses_dev, hbar_over_kb(), rec, recf, recn, occ, aux, evec, evecc, ph1d, qc, qmm, maxima, st);
    CU(cudaGetLastError());
    unsigned long long hmax[2] = {0, 0};
    CU(cudaMemcpyAsync(hmax, maxima, sizeof(hmax), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    {   // FP32 pre-filter constants: every candidate the pinned FP64 decision allows satisfies
        //   Delta_f^2 <= pfK1 * |u_a - u_b|_f^2 + pfC2   in FP32 arithmetic on the FP32-rounded table.
        double omax, umax;
        std::memcpy(&omax, &hmax[0], 8); std::memcpy(&umax, &hmax[1], 8);
        const double eta = 1e-2;                                      // 2 delta r <= eta r^2 + delta^2/eta
        const double da = 1e-6 * omax;                                // |Delta_f - Delta|  (bound 6.6e-7 omega_max)
        double K1, C2;
        if (d.sigma_const > 0.0) {
            const double r = d.ncut * d.sigma_const * (1.0 + 1e-6) + da;
            K1 = 0.0; C2 = r * r * (1.0 + 1e-5);
        } else {
            const double cs = d.ncut * d.scale / std::sqrt(6.0);
            const double dr = cs * 1e-6 * umax;                       // | |u_a-u_b|_f - |u_a-u_b| | (bound 4.2e-7 u_max)
            const double dd = da + dr;
            K1 = cs * cs * (1.0 + eta + 1e-5); C2 = dd * dd * (1.0 + 1.0 / eta) * (1.0 + 1e-5);
        }
        if (!(K1 < 1e30) || !(C2 < 1e30)) { K1 = 0.0; C2 = INFINITY; }  // filter disabled (ncut = inf): admit everything
        // upper bound of every entry of the stage 1 table (same formula as k_tables, rounded up once more)
        const double nmax = (d.sigma_const > 0.0 ? d.pfCs : d.pfCs * umax) * (1.0 + 2e-6) + d.pfSlack;
        d.pfNmax = std::isfinite(nmax) ? std::nextafterf((float)nmax, INFINITY) : INFINITY;
        // stage-1 tile test: |Delta_f| <= n'_a + n'_b <= 2 nmax, plus the rounding of the three FP32 adds of the bound
        d.pfW = std::isfinite(nmax) ? std::nextafterf((float)(2.0 * nmax + 1e-5 * wmax), INFINITY) : INFINITY;
        d.pfK1 = std::nextafterf((float)K1, INFINITY);
        d.pfC2 = std::isinf(C2) ? INFINITY : std::nextafterf((float)C2, INFINITY);
        // group path (k_enum_g): a pair (A, B) can hold an allowed process of a row only if the row's base energy lies
        // within bnd = gfC |u_a - u_b|_f + gfD of omega_B - s2 omega_A, all in FP32:
        //   ncut sigma = cs r,  r <= r_f + 2e-6 u_max (FP32 rounding of u, the subtraction, the squares, sqrt),
        //   the FP32 interval test is off by at most 8 eps omega_max + eps bnd < 1e-6 omega_max
        // (factors 1 + 1e-5: FP32 evaluation of the bound itself).
        const double cs = d.sigma_const > 0.0 ? 0.0 : d.ncut * d.scale / std::sqrt(6.0);
        const double half = d.sigma_const > 0.0 ? d.ncut * d.sigma_const * (1.0 + 1e-6) : 0.0;
        const double gd = (half + 1e-6 * omax + cs * 2e-6 * umax) * (1.0 + 1e-5);
        if (std::isfinite(cs) && std::isfinite(gd) && cs < 1e30 && gd < 1e30) {
            d.gfC = std::nextafterf((float)(cs * (1.0 + 1e-5)), INFINITY);
            d.gfD = std::nextafterf((float)gd, INFINITY);
            const double wmx = (double)d.gfC * 2.0 * umax * (1.0 + 1e-5) + (double)d.gfD + 1e-5 * omax;
            d.gfW = std::nextafterf((float)wmx, INFINITY);
        } else {                                                      // ncut = inf: every pair can hold every row
            d.gfC = 0.0f; d.gfD = INFINITY; d.gfW = INFINITY;
        }
        d.pfOff = 0;
        d.thrC = d.ncut * d.scale / std::sqrt(6.0);
        d.invC = d.sigma_const > 0.0 ? 1.0 / d.sigma_const : std::sqrt(6.0) / d.scale;
    }
    *out = ctx;
    return FP_OK;
#undef CU
#define CU(call)                                                                                         \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess)                                                                           \
            return fail(ctx, FP_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));              \
    } while (0)
}

int fp_destroy(fp_ctx *ctx) {
    if (!ctx) return FP_OK;
    for (auto &e : ctx->events) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
    for (auto &e : ctx->pool) cudaEventDestroy(e);
    for (int i = 0; i < 2; i++) {
        if (ctx->ev_enum[i]) cudaEventDestroy(ctx->ev_enum[i]);
        if (ctx->ev_eval[i]) cudaEventDestroy(ctx->ev_eval[i]);
    }
    if (ctx->side) cudaStreamDestroy(ctx->side);
    delete ctx;
    return FP_OK;
}

// ---- shared driver of fp_rates3 / fp_rates4 ------------------------------------------------------------------------------
// Rows (3ph: (target, channel); 4ph: (target, channel, lambda')) are independent: one launch of the fused kernel per
// super-chunk of targets whose per-row partial sums fit the scratch (Algorithm 5's bounded-memory loop, PAPER.md:354-393,
// with chunks of many modes instead of one), then the fixed-order per-mode reduction.
static int rates_driver(fp_ctx *ctx, int order, const int32_t *targets, int64_t nt, int32_t qp_begin, int32_t qp_end,
                        double *gamma, double *wp, int64_t *counts, fp_memloc loc, cudaStream_t st, bool reduce = true);

// Time reversal (fp_set_target_symmetry): evaluate one target of every {(q,j), (-q,j)} pair of the list and copy its
// rates, weighted phase space and counts to the other -- the sums of the two targets run over mirrored (q' -> -q')
// sets of processes with bitwise equal window decisions and weights and complex-conjugate matrix elements.  Only for
// whole q' ranges (a partial range of one target is the mirrored range of the other).
static int rates_reduced(fp_ctx *ctx, int order, const std::vector<int32_t> &ht, int32_t qp_begin, int32_t qp_end, double *gamma,
                         double *wp, int64_t *counts, fp_memloc loc, cudaStream_t st, bool &done) {
    const FpDev &d = ctx->d;
    const int64_t nt = (int64_t)ht.size();
    const int nch = order == 3 ? 2 : 3;
    done = false;
    std::map<int32_t, int32_t> slot;                                  // representative mode -> index into reps
    std::vector<int32_t> reps, where(nt);
    for (int64_t i = 0; i < nt; i++) {
        const int32_t q = ht[i] / d.nb, j = ht[i] - q * d.nb;
        const int32_t r = std::min(q, ctx->qpartner[q]) * d.nb + j;
        auto it = slot.find(r);
        if (it == slot.end()) { it = slot.emplace(r, (int32_t)reps.size()).first; reps.push_back(r); }
        where[i] = it->second;
    }
    if ((int64_t)reps.size() == nt) return FP_OK;                     // nothing to share: the caller runs the plain path
    const size_t nr = reps.size();
    std::vector<double> g(nr * nch), w(nr * nch), go(nt * nch), wo(nt * nch);
    std::vector<int64_t> c(nr * nch), co(nt * nch);
    int rc = rates_driver(ctx, order, reps.data(), (int64_t)nr, qp_begin, qp_end, g.data(), w.data(), c.data(), FP_MEM_HOST, st, false);
    if (rc != FP_OK) return rc;
    for (int64_t i = 0; i < nt; i++)
        for (int k = 0; k < nch; k++) {
            go[i * nch + k] = g[(size_t)where[i] * nch + k]; wo[i * nch + k] = w[(size_t)where[i] * nch + k];
            co[i * nch + k] = c[(size_t)where[i] * nch + k];
        }
    if (ctx->profiling) {                                             // processes delivered, not only those evaluated
        int64_t extra = 0;
        for (int64_t v : co) extra += v;
        for (int64_t v : c) extra -= v;
        ctx->prof.processes += extra;
    }
    const cudaMemcpyKind kind = loc == FP_MEM_HOST ? cudaMemcpyHostToHost : cudaMemcpyHostToDevice;
    CU(cudaMemcpyAsync(gamma, go.data(), go.size() * 8, kind, st));
    if (wp) CU(cudaMemcpyAsync(wp, wo.data(), wo.size() * 8, kind, st));
    if (counts) CU(cudaMemcpyAsync(counts, co.data(), co.size() * 8, kind, st));
    CU(cudaStreamSynchronize(st));
    done = true;
    return FP_OK;
}

static int rates_driver(fp_ctx *ctx, int order, const int32_t *targets, int64_t nt, int32_t qp_begin, int32_t qp_end,
                        double *gamma, double *wp, int64_t *counts, fp_memloc loc, cudaStream_t st, bool reduce) {
    if (!ctx) return FP_EINVAL;
    const FpDev &d = ctx->d;
    const IfcDev &f = order == 3 ? ctx->i3 : ctx->i4;
    if (!(order == 3 ? ctx->has3 : ctx->has4)) return fail(ctx, FP_ESTATE, "no IFC list of this order was given to fp_setup");
    if (nt < 0 || (nt > 0 && (!targets || !gamma))) return fail(ctx, FP_EINVAL, "null targets/gamma");
    if (order == 4 && (qp_begin < 0 || qp_end > d.N || qp_begin > qp_end)) return fail(ctx, FP_EINVAL, "bad q' range");
    if (nt == 0) return FP_OK;
    const int nch = order == 3 ? 2 : 3;
    const int64_t nqp = order == 3 ? 1 : (qp_end - qp_begin);
    const int64_t rows_per_unit = order == 3 ? 1 : nqp * d.nb;      // rows per (target, channel)
    const int64_t rows_per_target = nch * rows_per_unit;
    const int64_t nmodes = (int64_t)d.N * d.nb;
    const int64_t row_cands = (int64_t)d.N * d.nb * d.nb;

    // host copy of the targets for validation
    std::vector<int32_t> ht(nt);
    if (loc == FP_MEM_HOST) std::memcpy(ht.data(), targets, nt * sizeof(int32_t));
    else { CU(cudaMemcpyAsync(ht.data(), targets, nt * sizeof(int32_t), cudaMemcpyDeviceToHost, st)); CU(cudaStreamSynchronize(st)); }
    for (int64_t i = 0; i < nt; i++)
        if (ht[i] < 0 || ht[i] >= nmodes) return fail(ctx, FP_EINVAL, "target mode index out of range");

    if (reduce && ctx->trs_ok && ctx->use_trs && (order == 3 || (qp_begin == 0 && qp_end == d.N))) {
        bool done = false;
        const int rc = rates_reduced(ctx, order, ht, qp_begin, qp_end, gamma, wp, counts, loc, st, done);
        if (rc != FP_OK || done) return rc;
    }
    if (nqp == 0) {                                                   // empty q' range: all outputs zero
        std::vector<double> z(nt * nch, 0.0); std::vector<int64_t> zc(nt * nch, 0);
        cudaMemcpyKind k = loc == FP_MEM_HOST ? cudaMemcpyHostToHost : cudaMemcpyHostToDevice;
        CU(cudaMemcpyAsync(gamma, z.data(), z.size() * 8, k, st));
        if (wp) CU(cudaMemcpyAsync(wp, z.data(), z.size() * 8, k, st));
        if (counts) CU(cudaMemcpyAsync(counts, zc.data(), zc.size() * 8, k, st));
        CU(cudaStreamSynchronize(st));
        return FP_OK;
    }
    // The level-1 table of a row (nblk x 9 complex numbers, 144 bytes per contraction block) lives in shared memory: with
    // the queues of the fused kernel that caps the list at about 1,400 blocks (include/fourphonon.h, "Limits").
    auto too_many_blocks = [&](size_t need) {
        return fail(ctx, FP_ENOMEM, "IFC" + std::to_string(order) + " list has " + std::to_string(f.nblk) + " contraction blocks (atomA, atomB, dR): "
                    "its per-row table needs " + std::to_string(need) + " bytes of shared memory, more than the 226 KB of one SM "
                    "(limit about 1,400 blocks)");
    };
    // ... except for IFC3, whose Mhat is the level-0 table itself: past the limit the 3ph kernels read it from global memory
    const bool mg = ifc_mglobal(d, f, order);
    if (rates_smem_bytes(d, f, mg) > 227 * 1024 - 1024) return too_many_blocks(rates_smem_bytes(d, f, mg));

    // ---- scratch budget: per-target arrays for a super-chunk of targets ------------------------------------------------
    const size_t scratch_all = ctx->ws_bytes - ctx->resident;
    // ---- path: group path (lists in the scratch) when half of the scratch holds the list slots of a few hundred rows ----
    // list slot of one (row, warp): a quarter of what can never overflow (but at least 2048 entries); a group with a
    // slot that fills up is flagged by k_enum_g and its rows are redone through the fused kernel (rows of the many-branch
    // config 4, where the +- channel admits 10 % and more of the candidates; never on the diamond configs)
    const int64_t capw_all = enum_slot_entries(d);
    const int64_t capw = std::min(capw_all, std::max<int64_t>(((capw_all / FP_SLOT_DIV) + 31) & ~(int64_t)31, 2048));
    const size_t row_list_bytes = (size_t)enum_units(d) * ((size_t)capw * sizeof(ListEnt) + sizeof(uint32_t));
    // Groups (fp_group.cu): targets of a super-chunk that share their q-point; the rows of a group CTA share one scan of
    // the two free legs.  An unbounded window (ncut = inf) queues every (pair, row): small groups keep the queue bounded.
    const size_t list_region = scratch_all / 2;
    const bool overlap = ctx->path == FP_PATH_SPLIT;
    const int nbuf = overlap ? 2 : 1;
    const int64_t rows_fit = (int64_t)(list_region / (nbuf * row_list_bytes));   // rows whose list slots fit one buffer
    // the queue of a warp holds FP_ENUM_QC survivors; an unbounded window (ncut = inf) queues every (pair, row)
    const int rcap = (int)std::max<int64_t>(1, std::min<int64_t>(std::isfinite(d.gfW) ? FP_GROUP_RMAX : 4, rows_fit));
    const int mcap = order == 3 ? std::min(rcap, d.nb) : std::max(1, rcap / d.nb);   // members (targets) of a group
    const int njcap = order == 3 ? 1 : std::min(rcap, d.nb);        // j' of a 4ph group (all of them unless memory is short)
    const int rbound = order == 3 ? mcap : mcap * njcap;             // rows of a group, at most
    // FP_PATH_SPLIT runs the enumerator of chunk k+1 beside the evaluator of chunk k (two list buffers, two streams);
    // FP_PATH_SPLIT_SERIAL -- what FP_PATH_AUTO picks -- runs them back to back through one buffer of twice the groups.
    const int64_t rows_wanted = std::min<int64_t>(nt * nch * rows_per_unit, 256);
    bool split = ctx->path == FP_PATH_SPLIT || ctx->path == FP_PATH_SPLIT_SERIAL ||
                 (ctx->path == FP_PATH_AUTO && rows_fit >= rows_wanted);
    if (split && rows_fit < 1) return fail(ctx, FP_ENOMEM, "workspace scratch too small for the process lists of one row");
    if (split && !ctx->side) {
        int prio_lo = 0, prio_hi = 0;                                // enumerator CTAs take freed SM slots first: they need
        CU(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));    // few registers and keep the evaluator fed
        CU(cudaStreamCreateWithPriority(&ctx->side, cudaStreamNonBlocking, prio_hi));
        for (int i = 0; i < 2; i++) {
            CU(cudaEventCreateWithFlags(&ctx->ev_enum[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&ctx->ev_eval[i], cudaEventDisableTiming));
        }
    }
    // rows of one evaluator tile: their Mhat tables share the CTA's shared memory (FP_EVAL_TILE_BYTES of it)
    int ge = 1;
    if (split) {
        const size_t rowbytes = (size_t)f.nblk * 9 * sizeof(double2);
        ge = (int)std::max<size_t>(1, std::min<size_t>((size_t)rbound, FP_EVAL_TILE_BYTES / rowbytes));
        if (mg) ge = std::min(rbound, 6);                             // (no table in shared memory: the rows of one q-point)
        if (order == 4 && ge >= njcap) ge = ge / njcap * njcap;      // whole targets: their rows share the level-0 loads
        if (eval_smem_bytes(d, f, ge, mg) > 227 * 1024 - 1024) return too_many_blocks(eval_smem_bytes(d, f, ge, mg));
    }
    const size_t scratch = split ? scratch_all - list_region - 4096 : scratch_all;
    const size_t pre_per_target = (order == 3 ? (size_t)f.nblk * 9 : (size_t)f.n * 27) * sizeof(double2);
    const size_t per_target = pre_per_target + (size_t)rows_per_target * (4 + 16) + (size_t)nch * 24 + 4 + 64 + 16 +
                              (order == 4 ? (size_t)d.nb * 16 : 16);   // (+ group descriptors)
    const size_t fixed = 16 * 1024;
    if (scratch < fixed + per_target) return fail(ctx, FP_ENOMEM, "workspace scratch too small for one target");
    int64_t nts_max = (int64_t)std::min<size_t>((size_t)nt, (scratch - fixed) / per_target);
    while (nts_max * rows_per_target > (int64_t)1 << 30) nts_max = std::max<int64_t>(1, nts_max / 2);

    const double c_over_n = order == 3 ? const_c3() / (double)d.N : const_c4() / ((double)d.N * (double)d.N);

    for (int64_t t0 = 0; t0 < nt; t0 += nts_max) {
        const int64_t nts = std::min(nts_max, nt - t0);
        const int64_t nrows = nts * rows_per_target;
        Bump sc{ctx->ws, ctx->resident, ctx->ws_bytes};
        int32_t *d_targets = nullptr;
        if (loc == FP_MEM_DEVICE) d_targets = const_cast<int32_t *>(targets) + t0;
        else {
            d_targets = sc.take<int32_t>(nts);
            if (!d_targets) return fail(ctx, FP_ENOMEM, "scratch");
            CU(cudaMemcpyAsync(d_targets, targets + t0, nts * sizeof(int32_t), cudaMemcpyHostToDevice, st));
        }
        double2 *pre = sc.take<double2>(nts * (pre_per_target / sizeof(double2)));
        uint32_t *cnt = sc.take<uint32_t>(nrows);
        double2 *partial = sc.take<double2>(nrows);
        unsigned long long *stat = sc.take<unsigned long long>(5);    // [0] pre-filter survivors, [1] list overflows, [2] list entries, [3], [4] work counters
        double *o_gamma = sc.take<double>(nts * nch), *o_wp = sc.take<double>(nts * nch);
        int64_t *o_cnt = sc.take<int64_t>(nts * nch);
        if (!pre || !cnt || !partial || !stat || !o_gamma || !o_wp || !o_cnt) return fail(ctx, FP_ENOMEM, "scratch");

        RowArgs ra; ra.targets = d_targets; ra.row0 = 0; ra.qp_begin = qp_begin; ra.nqp = (int)nqp;
        ra.prefiltered = ctx->profiling ? stat : nullptr;
        ra.overflow = reinterpret_cast<unsigned int *>(stat + 1);
        ra.evaluated = ctx->profiling ? stat + 2 : nullptr;
        ra.sym = 0;
        ra.mglobal = mg ? 1 : 0;
        const int use_sym = (split && ctx->use_sym && (order == 4 ? ctx->sym34 : ctx->sym23)) ? 1 : 0;
        CU(cudaMemsetAsync(stat, 0, 3 * sizeof(unsigned long long), st));
        { ProfScope p(ctx, CAT_PRE, st);
          if (order == 3) launch_pre3(d, f, d_targets, nts, pre, st); else launch_pre4(d, f, d_targets, nts, pre, st); }
        CU(cudaGetLastError());
        // groups: the targets of this super-chunk sorted by q-point (stable), cut where q changes or at mcap members
        std::vector<int4> hgd;
        std::vector<int32_t> hgmem(nts);
        if (!split) {
            ProfScope p(ctx, CAT_RATES, st);
            CU(launch_rates(order, d, f, ra, nrows, pre, partial, cnt, false, st));
        } else {
            int rmaxg = 1;
            {
                std::vector<int32_t> ord(nts);
                for (int64_t i = 0; i < nts; i++) ord[i] = (int32_t)i;
                std::stable_sort(ord.begin(), ord.end(), [&](int32_t x, int32_t y) { return ht[t0 + x] / d.nb < ht[t0 + y] / d.nb; });
                for (int64_t i = 0; i < nts; i++) hgmem[i] = ord[i];
                for (int64_t i = 0; i < nts;) {
                    const int32_t q = ht[t0 + ord[i]] / d.nb;
                    int64_t e = i + 1;
                    while (e < nts && e - i < mcap && ht[t0 + ord[e]] / d.nb == q) e++;
                    if (order == 3) hgd.push_back(make_int4(q, (int)i, (int)(e - i), 0 | (1 << 16)));
                    else
                        for (int j0 = 0; j0 < d.nb; j0 += njcap)
                            hgd.push_back(make_int4(q, (int)i, (int)(e - i), j0 | (std::min(njcap, d.nb - j0) << 16)));
                    rmaxg = std::max<int>(rmaxg, (int)(e - i) * (order == 3 ? 1 : njcap));
                    i = e;
                }
            }
            const int64_t ng = (int64_t)hgd.size();
            int4 *d_gd = sc.take<int4>(ng);
            int32_t *d_gmem = sc.take<int32_t>(nts);
            if (!d_gd || !d_gmem) return fail(ctx, FP_ENOMEM, "scratch (groups)");
            CU(cudaMemcpyAsync(d_gd, hgd.data(), ng * sizeof(int4), cudaMemcpyHostToDevice, st));
            CU(cudaMemcpyAsync(d_gmem, hgmem.data(), nts * sizeof(int32_t), cudaMemcpyHostToDevice, st));
            GroupArgs ga; ga.targets = d_targets; ga.gdesc = d_gd; ga.gmem = d_gmem;
            ga.ng = (int)ng; ga.rmaxg = rmaxg; ga.nu = enum_units(d); ga.qp_begin = qp_begin; ga.nqp = (int)nqp; ga.gid0 = 0; ga.sym = use_sym;
            ga.prefiltered = ra.prefiltered; ga.evaluated = ra.evaluated; ga.overflow = ra.overflow;
            const int64_t ngc = ng * nch * nqp;                       // group CTAs: (group, channel[, q'])
            const int64_t chunk_gc = std::min<int64_t>(ngc, (int64_t)(list_region / (nbuf * (size_t)rmaxg * row_list_bytes)));
            const int ge_t = std::min(ge, rmaxg);
            // chunks of group CTAs through one or two list buffers: with two, the enumerator of chunk k+1 (side stream) runs
            // beside the evaluator of chunk k (caller's stream); buffer b is rewritten only after the evaluator that read it
            // has finished
            ListEnt *lists[2]; uint32_t *wcnt[2];
            for (int b = 0; b < nbuf; b++) {
                lists[b] = sc.take<ListEnt>((size_t)chunk_gc * rmaxg * enum_units(d) * capw);
                wcnt[b] = sc.take<uint32_t>((size_t)chunk_gc * rmaxg * enum_units(d));
                if (!lists[b] || !wcnt[b]) return fail(ctx, FP_ENOMEM, "scratch (process lists)");
            }
            cudaStream_t es = overlap ? ctx->side : st;
            if (overlap) {                                           // targets, groups and statistics are ready on st
                CU(cudaEventRecord(ctx->ev_eval[0], st));
                CU(cudaStreamWaitEvent(es, ctx->ev_eval[0], 0));
            }
            int k = 0;
            for (int64_t g0 = 0; g0 < ngc; g0 += chunk_gc, k++) {
                const int64_t n = std::min(chunk_gc, ngc - g0);
                const int b = overlap ? (k & 1) : 0;
                GroupArgs gc = ga; gc.gid0 = g0;
                if (overlap && k >= 2) CU(cudaStreamWaitEvent(es, ctx->ev_eval[b], 0));
                { ProfScope p(ctx, CAT_ENUM, es);
                  CU(launch_enum_g(order, d, gc, n, capw, lists[b], wcnt[b], reinterpret_cast<unsigned int *>(stat + 3 + b), ctx->sm_count, es)); }
                if (overlap) {
                    CU(cudaEventRecord(ctx->ev_enum[b], es));
                    CU(cudaStreamWaitEvent(st, ctx->ev_enum[b], 0));
                }
                { ProfScope p(ctx, CAT_RATES, st);
                  CU(launch_eval_g(order, d, f, gc, n, pre, capw, lists[b], wcnt[b], ge_t, partial, cnt, ctx->precision == FP_PREC_MIXED, mg, st)); }
                if (overlap) CU(cudaEventRecord(ctx->ev_eval[b], st));
            }
            unsigned long long novf = 0;
            CU(cudaMemcpyAsync(&novf, stat + 1, sizeof(novf), cudaMemcpyDeviceToHost, st));
            CU(cudaStreamSynchronize(st));
            if (novf != 0) {                                         // some groups gave up (a list slot or the survivor queue
                ctx->prof.list_overflows += (int64_t)novf;           // filled up): k_eval_g marked their rows in cnt; redo those
                RowArgs rr = ra; rr.prefiltered = nullptr;           // with the lists in shared memory
                ProfScope p(ctx, CAT_RATES, st);
                CU(launch_rates(order, d, f, rr, nrows, pre, partial, cnt, true, st));
            }
        }
        double *g_out = loc == FP_MEM_DEVICE ? gamma + t0 * nch : o_gamma;
        double *w_out = (loc == FP_MEM_DEVICE && wp) ? wp + t0 * nch : o_wp;
        int64_t *c_out = (loc == FP_MEM_DEVICE && counts) ? counts + t0 * nch : o_cnt;
        { ProfScope p(ctx, CAT_REDUCE, st);
          launch_finalize(order, d, nts, rows_per_unit, partial, cnt, c_over_n, g_out, w_out, c_out, st); }
        CU(cudaGetLastError());
        if (loc == FP_MEM_HOST) {
            CU(cudaMemcpyAsync(gamma + t0 * nch, g_out, nts * nch * 8, cudaMemcpyDeviceToHost, st));
            if (wp) CU(cudaMemcpyAsync(wp + t0 * nch, w_out, nts * nch * 8, cudaMemcpyDeviceToHost, st));
            if (counts) CU(cudaMemcpyAsync(counts + t0 * nch, c_out, nts * nch * 8, cudaMemcpyDeviceToHost, st));
        }
        CU(cudaStreamSynchronize(st));                               // the scratch is reused by the next super-chunk
        if (ctx->profiling) {                                        // analytic models, DESIGN.md §6
            std::vector<int64_t> hc(nts * nch);
            unsigned long long hstat3[3] = {0, 0, 0};
            CU(cudaMemcpy(hc.data(), c_out, nts * nch * 8, cudaMemcpyDeviceToHost));
            CU(cudaMemcpy(hstat3, stat, sizeof(hstat3), cudaMemcpyDeviceToHost));
            const unsigned long long hstat = hstat3[0];
            int64_t total = 0;
            for (int64_t v : hc) total += v;
            ctx->prof.rows += nrows;
            ctx->prof.processes += total;
            ctx->prof.prefiltered += (int64_t)hstat;
            ctx->prof.candidates += nrows * row_cands;
            // matrix elements evaluated: the list entries of the split path (rows redone by k_rates after a list overflow
            // are not in this figure), else one per process
            const int64_t evaluated = split ? (int64_t)hstat3[2] : total;
            ctx->prof.evaluated += evaluated;
            ctx->prof.rates_flops += (double)evaluated * (order == 3 ? ctx->flops_elem3 : ctx->flops_elem4);
        }
    }
    return FP_OK;
}

int fp_rates3(fp_ctx *ctx, const int32_t *targets, int64_t ntargets, double *gamma, double *wp, int64_t *counts,
              fp_memloc loc, void *stream) {
    return rates_driver(ctx, 3, targets, ntargets, 0, 1, gamma, wp, counts, loc, (cudaStream_t)stream);
}

int fp_rates4(fp_ctx *ctx, const int32_t *targets, int64_t ntargets, int32_t qp_begin, int32_t qp_end, double *gamma,
              double *wp, int64_t *counts, fp_memloc loc, void *stream) {
    return rates_driver(ctx, 4, targets, ntargets, qp_begin, qp_end, gamma, wp, counts, loc, (cudaStream_t)stream);
}

int fp_kappa_rta(fp_ctx *ctx, const double *gamma_total, double *kappa, fp_memloc loc, void *stream) {
    if (!ctx || !gamma_total || !kappa) return ctx ? fail(ctx, FP_EINVAL, "null argument") : FP_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const FpDev &d = ctx->d;
    const size_t M = (size_t)d.N * d.nb;
    const double pref = const_ckappa() / (d.T * d.T * ctx->vol * (double)d.N);
    if (loc == FP_MEM_DEVICE) {
        launch_kappa(d, gamma_total, pref, kappa, st);
        CU(cudaGetLastError());
        return FP_OK;
    }
    Bump sc{ctx->ws, ctx->resident, ctx->ws_bytes};
    double *g = sc.take<double>(M), *k = sc.take<double>(9);
    if (!g || !k) return fail(ctx, FP_ENOMEM, "scratch");
    CU(cudaMemcpyAsync(g, gamma_total, M * 8, cudaMemcpyHostToDevice, st));
    launch_kappa(d, g, pref, k, st);
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(kappa, k, 72, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return FP_OK;
}

// ---- debug list export -------------------------------------------------------------------------------------------------
static int list_driver(fp_ctx *ctx, int order, int32_t target, int32_t channel, int32_t qp, int32_t *out, int64_t cap,
                       int64_t *n, cudaStream_t st, double *terms = nullptr) {
    if (!ctx || !n) return FP_EINVAL;
    const FpDev &d = ctx->d;
    if (!(order == 3 ? ctx->has3 : ctx->has4)) return fail(ctx, FP_ESTATE, "no IFC list of this order was given to fp_setup");
    const int nch = order == 3 ? 2 : 3;
    if (target < 0 || target >= d.N * d.nb || channel < 0 || channel >= nch || cap < 0 || (cap > 0 && !out))
        return fail(ctx, FP_EINVAL, "bad target/channel/cap");
    if (order == 4 && (qp < 0 || qp >= d.N)) return fail(ctx, FP_EINVAL, "bad q'");
    const int64_t rows_per_unit = order == 3 ? 1 : d.nb;
    const int64_t nrows = nch * rows_per_unit;
    const int w = order == 3 ? 2 : 3;
    Bump sc{ctx->ws, ctx->resident, ctx->ws_bytes};
    int32_t *d_t = sc.take<int32_t>(1);
    uint32_t *cnt = sc.take<uint32_t>(nrows);
    int64_t *offs = sc.take<int64_t>(nrows + 1), *bsums = sc.take<int64_t>(16);
    if (!d_t || !cnt || !offs || !bsums) return fail(ctx, FP_ENOMEM, "scratch");
    CU(cudaMemcpyAsync(d_t, &target, 4, cudaMemcpyHostToDevice, st));
    RowArgs ra; ra.targets = d_t; ra.row0 = 0; ra.qp_begin = qp; ra.nqp = 1; ra.prefiltered = nullptr; ra.overflow = nullptr;
    ra.evaluated = nullptr; ra.sym = 0;
    ra.mglobal = ifc_mglobal(d, order == 3 ? ctx->i3 : ctx->i4, order) ? 1 : 0;
    launch_count(order, d, ra, nrows, cnt, st);
    launch_scan(cnt, nrows, offs, bsums, st);
    std::vector<int64_t> ho(nrows + 1);
    CU(cudaMemcpyAsync(ho.data(), offs, (nrows + 1) * 8, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    const int64_t total = ho[nrows];
    uint32_t *list = sc.take<uint32_t>(std::max<int64_t>(total, 1));
    int32_t *dec = sc.take<int32_t>(std::max<int64_t>(total, 1) * w);
    if (!list || !dec) return fail(ctx, FP_ENOMEM, "scratch");
    launch_fill(order, d, ra, nrows, offs, 0, list, st);
    const int64_t rb = channel * rows_per_unit, re = rb + rows_per_unit;
    for (int64_t r = rb; r < re; r++) {
        RowArgs rr = ra; rr.row0 = r;
        launch_decode(order, d, rr, list + ho[r], ho[r + 1] - ho[r], dec + (ho[r] - ho[rb]) * w, st);
    }
    CU(cudaGetLastError());
    *n = ho[re] - ho[rb];
    const int64_t ncopy = std::min(*n, cap);
    if (ncopy > 0) CU(cudaMemcpyAsync(out, dec, ncopy * w * 4, cudaMemcpyDeviceToHost, st));
    if (terms && *n > 0) {                                            // per-process terms: level 0 of the target, then k_terms
        const IfcDev &f = order == 3 ? ctx->i3 : ctx->i4;
        if (rates_smem_bytes(d, f, ra.mglobal != 0) > 227 * 1024 - 1024) return fail(ctx, FP_ENOMEM, "IFC block table exceeds the shared memory of one SM");
        double2 *pre = sc.take<double2>(order == 3 ? (size_t)f.nblk * 9 : (size_t)f.n * 27);
        double *gp = sc.take<double>(*n);
        if (!pre || !gp) return fail(ctx, FP_ENOMEM, "scratch");
        if (order == 3) launch_pre3(d, f, d_t, 1, pre, st); else launch_pre4(d, f, d_t, 1, pre, st);
        const double sym = order == 3 ? (channel == 0 ? 1.0 : 0.5) : (channel == 2 ? 1.0 / 6.0 : 0.5);
        const double c_over_n = order == 3 ? const_c3() / (double)d.N : const_c4() / ((double)d.N * (double)d.N);
        RowArgs rr = ra; rr.row0 = rb;
        CU(launch_terms(order, d, f, rr, re - rb, pre, offs, ho[rb], list + ho[rb], c_over_n * sym, gp, st));
        if (ncopy > 0) CU(cudaMemcpyAsync(terms, gp, ncopy * 8, cudaMemcpyDeviceToHost, st));
    }
    CU(cudaStreamSynchronize(st));
    return FP_OK;
}

int fp_list3(fp_ctx *ctx, int32_t target, int32_t channel, int32_t *pairs, int64_t cap, int64_t *n, void *stream) {
    return list_driver(ctx, 3, target, channel, 0, pairs, cap, n, (cudaStream_t)stream);
}
int fp_list4(fp_ctx *ctx, int32_t target, int32_t channel, int32_t qp, int32_t *triples, int64_t cap, int64_t *n,
             void *stream) {
    return list_driver(ctx, 4, target, channel, qp, triples, cap, n, (cudaStream_t)stream);
}

// ---- profiling ------------------------------------------------------------------------------------------------------------
int fp_set_path(fp_ctx *ctx, int path) {
    if (!ctx || path < FP_PATH_AUTO || path > FP_PATH_SPLIT_SERIAL) return ctx ? fail(ctx, FP_EINVAL, "unknown path") : FP_EINVAL;
    ctx->path = path;
    return FP_OK;
}

int fp_terms3(fp_ctx *ctx, int32_t target, int32_t channel, int32_t *pairs, double *gamma_p, int64_t cap, int64_t *n, void *stream) {
    if (!gamma_p && cap > 0) return ctx ? fail(ctx, FP_EINVAL, "null gamma_p") : FP_EINVAL;
    return list_driver(ctx, 3, target, channel, 0, pairs, cap, n, (cudaStream_t)stream, gamma_p);
}
int fp_terms4(fp_ctx *ctx, int32_t target, int32_t channel, int32_t qp, int32_t *triples, double *gamma_p, int64_t cap, int64_t *n,
              void *stream) {
    if (!gamma_p && cap > 0) return ctx ? fail(ctx, FP_EINVAL, "null gamma_p") : FP_EINVAL;
    return list_driver(ctx, 4, target, channel, qp, triples, cap, n, (cudaStream_t)stream, gamma_p);
}

int fp_set_symmetry(fp_ctx *ctx, int on) { if (!ctx) return FP_EINVAL; ctx->use_sym = on != 0; return FP_OK; }
int fp_get_symmetry(const fp_ctx *ctx) {
    return ctx ? ((ctx->use_sym && ctx->sym23 ? 1 : 0) | (ctx->use_sym && ctx->sym34 ? 2 : 0)) : FP_EINVAL;
}

int fp_set_precision(fp_ctx *ctx, int mode) {
    if (!ctx || (mode != FP_PREC_FP64 && mode != FP_PREC_MIXED)) return ctx ? fail(ctx, FP_EINVAL, "unknown precision mode") : FP_EINVAL;
    ctx->precision = mode;
    return FP_OK;
}
int fp_get_precision(const fp_ctx *ctx) { return ctx ? ctx->precision : FP_EINVAL; }

int fp_set_target_symmetry(fp_ctx *ctx, int on) { if (!ctx) return FP_EINVAL; ctx->use_trs = on != 0; return FP_OK; }
int fp_get_target_symmetry(const fp_ctx *ctx) { return ctx ? (ctx->use_trs && ctx->trs_ok ? 1 : 0) : FP_EINVAL; }

int fp_set_prefilter(fp_ctx *ctx, int on) {
    if (!ctx) return FP_EINVAL;
    FpDev &d = ctx->d;
    if (!on && !ctx->pf_saved) {                                      // every FP32 test admits everything that is not a zero mode
        ctx->sv_pfK1 = d.pfK1; ctx->sv_pfC2 = d.pfC2; ctx->sv_pfNmax = d.pfNmax; ctx->sv_pfW = d.pfW;
        ctx->sv_gfC = d.gfC; ctx->sv_gfD = d.gfD; ctx->sv_gfW = d.gfW;
        d.pfK1 = 0.0f; d.pfC2 = INFINITY; d.pfNmax = INFINITY; d.pfW = INFINITY;
        d.gfC = 0.0f; d.gfD = INFINITY; d.gfW = INFINITY;
        d.pfOff = 1;
        ctx->pf_saved = true;
    } else if (on && ctx->pf_saved) {
        d.pfK1 = ctx->sv_pfK1; d.pfC2 = ctx->sv_pfC2; d.pfNmax = ctx->sv_pfNmax; d.pfW = ctx->sv_pfW;
        d.gfC = ctx->sv_gfC; d.gfD = ctx->sv_gfD; d.gfW = ctx->sv_gfW;
        d.pfOff = 0;
        ctx->pf_saved = false;
    }
    return FP_OK;
}

int fp_profile_enable(fp_ctx *ctx, int on) { if (!ctx) return FP_EINVAL; ctx->profiling = on != 0; return FP_OK; }

int fp_profile_reset(fp_ctx *ctx) {
    if (!ctx) return FP_EINVAL;
    for (auto &e : ctx->events) { ctx->pool.push_back(e.a); ctx->pool.push_back(e.b); }
    ctx->events.clear();
    ctx->prof = fp_profile{};
    return FP_OK;
}

int fp_profile_get(fp_ctx *ctx, fp_profile *out) {
    if (!ctx || !out) return FP_EINVAL;
    fp_profile p = ctx->prof;
    p.ms_precontract = p.ms_rates = p.ms_reduce = p.ms_enum = 0;
    p.n_precontract = p.n_rates = p.n_reduce = p.n_enum = 0;
    for (auto &e : ctx->events) {
        CU(cudaEventSynchronize(e.b));
        float ms = 0;
        CU(cudaEventElapsedTime(&ms, e.a, e.b));
        switch (e.cat) {
            case CAT_PRE: p.ms_precontract += ms; p.n_precontract++; break;
            case CAT_RATES: p.ms_rates += ms; p.n_rates++; break;
            case CAT_REDUCE: p.ms_reduce += ms; p.n_reduce++; break;
            case CAT_ENUM: p.ms_enum += ms; p.n_enum++; break;
        }
    }
    *out = p;
    return FP_OK;
}

int fp_probe_fp64_tflops(void *stream, double *tflops) {
    if (!tflops) return FP_EINVAL;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return FP_ECUDA;
    double t = run_fp64_probe((cudaStream_t)stream, sms);
    if (t <= 0) return FP_ECUDA;
    *tflops = t;
    return FP_OK;
}

int fp_probe_dmma_tflops(void *stream, double out[3]) {
    if (!out) return FP_EINVAL;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return FP_ECUDA;
    run_dmma_probe((cudaStream_t)stream, sms, out);
    return (out[0] > 0 && out[1] > 0 && out[2] > 0) ? FP_OK : FP_ECUDA;
}

}  // extern "C"
